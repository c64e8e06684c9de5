// sort.cu -- periodic per-cell counting sort of one species (SURVEY 8(c.1)
// "Sort"; BASELINE.json:north_star part 5): key = i + nx*(j + ny*k) with
// (i,j,k) = clamp(floor(xi,eta,zeta)) of the stored position; histogram,
// exclusive scan, scatter of x,y,z,ux,uy,uz,w,id into the second SoA buffer.
// Integer work on 32-bit keys/counters (np < 2^31 is enforced at the ABI);
// fp64 payload is only moved.  HBM-bound: ~24 B read + 8 B written per
// particle for keys/ranks, 64 B read + 64 B written for the scatter.
#include "pic_internal.h"

namespace pic {

__device__ __forceinline__ int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

__global__ void __launch_bounds__(256) key_hist_kernel(Grid g, const double* __restrict__ x,
                                                       const double* __restrict__ y, const double* __restrict__ z,
                                                       long long n, unsigned int* __restrict__ key,
                                                       unsigned int* __restrict__ rank, unsigned int* count) {
    long long ip = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ip >= n) return;
    const int i = clampi(__double2int_rd((x[ip] - g.xmin) * g.inv_dx), 0, g.nx - 1);
    const int j = clampi(__double2int_rd((y[ip] - g.ymin) * g.inv_dy), 0, g.ny - 1);
    const int k = clampi(__double2int_rd((z[ip] - g.zmin) * g.inv_dz), 0, g.nz - 1);
    const unsigned int c = (unsigned int)i + (unsigned int)g.nx * ((unsigned int)j + (unsigned int)g.ny * (unsigned int)k);
    key[ip] = c;
    rank[ip] = atomicAdd(count + c, 1u);   // position inside the cell (order inside a cell is unspecified, R24)
}

// Keys already written by the fused particle kernel (it knows every particle's new cell): histogram and rank only,
// 4 B read + 4 B written per particle instead of 24 + 8.
__global__ void __launch_bounds__(256) hist_rank_kernel(long long n, const unsigned int* __restrict__ key,
                                                        unsigned int* __restrict__ rank, unsigned int* count) {
    long long ip = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ip >= n) return;
    // The keys arrive in the order of the last sort, so a warp holds a handful of distinct cells: one atomic per
    // distinct key and warp instead of one per particle (the kernel is bound by the rate of returned L2 atomics).
    const unsigned int k = key[ip];
    const unsigned int active = __activemask();
    const unsigned int same = __match_any_sync(active, k);
    const int leader = __ffs(same) - 1, lane = threadIdx.x & 31;
    unsigned int base = 0;
    if (lane == leader) base = atomicAdd(count + k, (unsigned int)__popc(same));
    base = __shfl_sync(same, base, leader);
    rank[ip] = base + (unsigned int)__popc(same & ((1u << lane) - 1u));
}

constexpr int SCAN_T = 256, SCAN_V = 8, SCAN_ITEMS = SCAN_T * SCAN_V;

// exclusive scan of each SCAN_ITEMS chunk in place; chunk totals to sums[]
__global__ void __launch_bounds__(SCAN_T) scan_chunks_kernel(unsigned int* data, long long n, unsigned int* sums) {
    __shared__ unsigned int warp_tot[SCAN_T / 32];
    const long long base = (long long)blockIdx.x * SCAN_ITEMS + (long long)threadIdx.x * SCAN_V;
    unsigned int v[SCAN_V];
    unsigned int tot = 0;
#pragma unroll
    for (int e = 0; e < SCAN_V; ++e) {
        v[e] = (base + e < n) ? data[base + e] : 0u;
        tot += v[e];
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    unsigned int inc = tot;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        unsigned int t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) warp_tot[wid] = inc;
    __syncthreads();
    unsigned int woff = 0, btot = 0;
#pragma unroll
    for (int w = 0; w < SCAN_T / 32; ++w) {
        if (w < wid) woff += warp_tot[w];
        btot += warp_tot[w];
    }
    unsigned int run = woff + inc - tot;
#pragma unroll
    for (int e = 0; e < SCAN_V; ++e) {
        if (base + e < n) data[base + e] = run;
        run += v[e];
    }
    if (threadIdx.x == 0) sums[blockIdx.x] = btot;
}

// exclusive scan of the chunk totals by one block
__global__ void __launch_bounds__(1024) scan_sums_kernel(unsigned int* sums, long long nb) {
    __shared__ unsigned int part[1024];
    const long long per = (nb + 1023) / 1024;
    const long long lo = (long long)threadIdx.x * per, hi = (lo + per < nb) ? lo + per : nb;
    unsigned int tot = 0;
    for (long long e = lo; e < hi; ++e) tot += sums[e];
    part[threadIdx.x] = tot;
    __syncthreads();
    // Hillis-Steele inclusive scan over 1024 partials
    for (int d = 1; d < 1024; d <<= 1) {
        unsigned int t = (threadIdx.x >= d) ? part[threadIdx.x - d] : 0u;
        __syncthreads();
        part[threadIdx.x] += t;
        __syncthreads();
    }
    unsigned int run = part[threadIdx.x] - tot;
    for (long long e = lo; e < hi; ++e) {
        unsigned int s = sums[e];
        sums[e] = run;
        run += s;
    }
}

__global__ void __launch_bounds__(SCAN_T) add_sums_kernel(unsigned int* data, long long n, const unsigned int* sums) {
    const long long base = (long long)blockIdx.x * SCAN_ITEMS + (long long)threadIdx.x * SCAN_V;
    const unsigned int off = sums[blockIdx.x];
#pragma unroll
    for (int e = 0; e < SCAN_V; ++e)
        if (base + e < n) data[base + e] += off;
}

__global__ void __launch_bounds__(256) scatter_kernel(Particles src, Particles dst, long long n,
                                                      const unsigned int* __restrict__ key,
                                                      const unsigned int* __restrict__ rank,
                                                      const unsigned int* __restrict__ offset) {
    long long ip = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ip >= n) return;
    const long long d = (long long)offset[key[ip]] + rank[ip];
    dst.x[d] = src.x[ip];
    dst.y[d] = src.y[ip];
    dst.z[d] = src.z[ip];
    dst.ux[d] = src.ux[ip];
    dst.uy[d] = src.uy[ip];
    dst.uz[d] = src.uz[ip];
    dst.w[d] = src.w[ip];
    dst.id[d] = src.id[ip];
}

// Deferred sort: only the permutation is written, perm[d] = index in the unsorted buffer of the particle that
// belongs at sorted position d (4 B per particle instead of 64 B read + 64 B written); the next fused particle
// kernel reads its inputs through it and writes its outputs in sorted order into the other buffer.
__global__ void __launch_bounds__(256) perm_kernel(long long n, const unsigned int* __restrict__ key,
                                                   const unsigned int* __restrict__ rank,
                                                   const unsigned int* __restrict__ offset,
                                                   unsigned int* __restrict__ perm) {
    long long ip = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ip >= n) return;
    perm[(long long)offset[key[ip]] + rank[ip]] = (unsigned int)ip;
}

// dst[d] = src[perm[d]] for every array (materialises a deferred sort for callers other than the tile kernel)
__global__ void __launch_bounds__(256) apply_perm_kernel(Particles src, Particles dst, long long n,
                                                         const unsigned int* __restrict__ perm) {
    long long d = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (d >= n) return;
    const long long ip = perm[d];
    dst.x[d] = src.x[ip];
    dst.y[d] = src.y[ip];
    dst.z[d] = src.z[ip];
    dst.ux[d] = src.ux[ip];
    dst.uy[d] = src.uy[ip];
    dst.uz[d] = src.uz[ip];
    dst.w[d] = src.w[ip];
    dst.id[d] = src.id[ip];
}

void launch_apply_perm(const Particles& src, const Particles& dst, long long n, const unsigned int* perm,
                       cudaStream_t st) {
    if (n > 0) apply_perm_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(src, dst, n, perm);
}

long long sort_block_sums_len(long long ncell) { return (ncell + 1 + SCAN_ITEMS - 1) / SCAN_ITEMS + 1; }

// perm == nullptr: scatter src -> dst now; else write the permutation only (src stays as it is, dst untouched)
// keys_in != nullptr: the cell keys of src as written by the last fused particle kernel
int launch_sort(const Grid& g, const Particles& src, const Particles& dst, long long n, unsigned int* cell_offset,
                unsigned int* perm, const unsigned int* keys_in, const SortScratch& sc, cudaStream_t st) {
    const long long ncell = (long long)g.nx * g.ny * g.nz;
    const long long nscan = ncell + 1;
    int launches = 0;
    const unsigned int* key = keys_in ? keys_in : sc.key;
    cudaMemsetAsync(cell_offset, 0, (size_t)nscan * sizeof(unsigned int), st);
    if (n > 0) {
        if (keys_in) hist_rank_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, keys_in, sc.rank, cell_offset);
        else key_hist_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(g, src.x, src.y, src.z, n, sc.key, sc.rank,
                                                                          cell_offset);
        ++launches;
    }
    const long long nb = (nscan + SCAN_ITEMS - 1) / SCAN_ITEMS;
    scan_chunks_kernel<<<(unsigned)nb, SCAN_T, 0, st>>>(cell_offset, nscan, sc.block_sums);
    scan_sums_kernel<<<1, 1024, 0, st>>>(sc.block_sums, nb);
    add_sums_kernel<<<(unsigned)nb, SCAN_T, 0, st>>>(cell_offset, nscan, sc.block_sums);
    launches += 3;
    if (n > 0) {
        if (perm) perm_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, key, sc.rank, cell_offset, perm);
        else scatter_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(src, dst, n, key, sc.rank, cell_offset);
        ++launches;
    }
    return launches;
}

}  // namespace pic
