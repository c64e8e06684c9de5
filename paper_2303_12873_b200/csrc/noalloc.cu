// noalloc.cu -- pic_cell_offsets_noalloc (include/pic_noalloc.h): the histogram + exclusive scan of the counting
// sort (SURVEY 8(c.1) "Sort") for callers that may not allocate device memory -- a hook inside another code's
// time loop whose pool owns all of HBM, a step where cudaMalloc's device-wide synchronisation is unaffordable, a
// diagnostic on an out-of-memory path.  Same arithmetic as sort.cu's key_hist / scan kernels, so the offsets are
// bit-identical to pic_sort's; the difference is where the scan's chunk totals live: not in the caller's arena
// but in the file-scope device array below, which belongs to the library image (64 KiB on every GPU that loads
// it, until the process exits).  Nothing here calls cudaMalloc, cudaFree or an allocating library routine.
//
// This file is self-contained on purpose: it shares no kernel with sort.cu, so the arena-based path is untouched.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>

#include <mutex>

#include "../../include/pic.h"
#include "../../include/pic_noalloc.h"

namespace {

constexpr int CHUNK_T = 256, CHUNK_V = 8, CHUNK = CHUNK_T * CHUNK_V;   // 2,048 counters per block, as pic_noalloc.h states
static_assert(CHUNK == 2048, "pic_noalloc.h quotes 2,048 counters per chunk");

// The scratch: one total per chunk.  In HOST code this name is only a stand-in the runtime uses to find the
// array; it is not a device address.  Host code below obtains the address with cudaGetSymbolAddress, once per
// device, and hands that pointer to the kernels.
static __device__ __align__(256) unsigned int g_chunk_totals[PIC_NOALLOC_MAX_CHUNKS];

constexpr int MAX_DEVICES = 64;
unsigned int* s_totals_on_device[MAX_DEVICES];   // device address of g_chunk_totals per device ordinal, 0 = not looked up yet
std::mutex s_setup_lock;
thread_local char t_error[256] = "";

int fail(int code, const char* what, cudaError_t e = cudaSuccess) {
    if (e != cudaSuccess) snprintf(t_error, sizeof t_error, "pic_cell_offsets_noalloc: %s: %s", what, cudaGetErrorString(e));
    else snprintf(t_error, sizeof t_error, "pic_cell_offsets_noalloc: %s", what);
    return code;
}

struct Box {
    int nx, ny, nz;
    double xmin, ymin, zmin, inv_dx, inv_dy, inv_dz;
};

__device__ __forceinline__ int clamp_cell(int v, int hi) { return v < 0 ? 0 : (v > hi ? hi : v); }

// count[c] += 1 for the cell c of every particle; a warp issues one atomic per distinct cell it holds
__global__ void __launch_bounds__(256) cell_count_kernel(Box b, const double* __restrict__ x, const double* __restrict__ y,
                                                         const double* __restrict__ z, long long n, unsigned int* count) {
    const long long ip = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ip >= n) return;
    const int i = clamp_cell(__double2int_rd((x[ip] - b.xmin) * b.inv_dx), b.nx - 1);
    const int j = clamp_cell(__double2int_rd((y[ip] - b.ymin) * b.inv_dy), b.ny - 1);
    const int k = clamp_cell(__double2int_rd((z[ip] - b.zmin) * b.inv_dz), b.nz - 1);
    const unsigned int c = (unsigned int)i + (unsigned int)b.nx * ((unsigned int)j + (unsigned int)b.ny * (unsigned int)k);
    const unsigned int same = __match_any_sync(__activemask(), c);
    if ((int)(threadIdx.x & 31) == __ffs(same) - 1) atomicAdd(count + c, (unsigned int)__popc(same));
}

// exclusive scan inside each chunk, in place; the chunk's total goes to totals[blockIdx.x]
__global__ void __launch_bounds__(CHUNK_T) chunk_scan_kernel(unsigned int* data, long long n, unsigned int* totals) {
    __shared__ unsigned int warp_sum[CHUNK_T / 32];
    const long long first = (long long)blockIdx.x * CHUNK + (long long)threadIdx.x * CHUNK_V;
    unsigned int v[CHUNK_V], mine = 0;
#pragma unroll
    for (int e = 0; e < CHUNK_V; ++e) {
        v[e] = (first + e < n) ? data[first + e] : 0u;
        mine += v[e];
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned int incl = mine;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned int up = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += up;
    }
    if (lane == 31) warp_sum[warp] = incl;
    __syncthreads();
    unsigned int before = 0, all = 0;
#pragma unroll
    for (int w = 0; w < CHUNK_T / 32; ++w) {
        if (w < warp) before += warp_sum[w];
        all += warp_sum[w];
    }
    unsigned int run = before + incl - mine;
#pragma unroll
    for (int e = 0; e < CHUNK_V; ++e) {
        if (first + e < n) data[first + e] = run;
        run += v[e];
    }
    if (threadIdx.x == 0) totals[blockIdx.x] = all;
}

// exclusive scan of the nchunks totals by one block (nchunks <= PIC_NOALLOC_MAX_CHUNKS = 16 per thread at most)
__global__ void __launch_bounds__(1024) totals_scan_kernel(unsigned int* totals, int nchunks) {
    __shared__ unsigned int part[1024];
    const int per = (nchunks + 1023) / 1024;
    const int lo = min((int)threadIdx.x * per, nchunks), hi = min(lo + per, nchunks);
    unsigned int mine = 0;
    for (int e = lo; e < hi; ++e) mine += totals[e];
    part[threadIdx.x] = mine;
    __syncthreads();
    for (int d = 1; d < 1024; d <<= 1) {
        const unsigned int t = ((int)threadIdx.x >= d) ? part[threadIdx.x - d] : 0u;
        __syncthreads();
        part[threadIdx.x] += t;
        __syncthreads();
    }
    unsigned int run = part[threadIdx.x] - mine;
    for (int e = lo; e < hi; ++e) {
        const unsigned int t = totals[e];
        totals[e] = run;
        run += t;
    }
}

__global__ void __launch_bounds__(CHUNK_T) add_totals_kernel(unsigned int* data, long long n, const unsigned int* totals) {
    const long long first = (long long)blockIdx.x * CHUNK + (long long)threadIdx.x * CHUNK_V;
    const unsigned int off = totals[blockIdx.x];
#pragma unroll
    for (int e = 0; e < CHUNK_V; ++e)
        if (first + e < n) data[first + e] += off;
}

// Device address of g_chunk_totals on the current device; looked up on the first call per device.
int scratch_on_current_device(unsigned int** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(PIC_ECUDA, "cudaGetDevice", e);
    if (dev < 0 || dev >= MAX_DEVICES) return fail(PIC_EINVAL, "device ordinal beyond 63");
    std::lock_guard<std::mutex> hold(s_setup_lock);
    if (!s_totals_on_device[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_chunk_totals);   // the address on the CURRENT device
        if (e != cudaSuccess || !p) return fail(PIC_ECUDA, "cudaGetSymbolAddress(g_chunk_totals)", e);
        s_totals_on_device[dev] = static_cast<unsigned int*>(p);
    }
    *out = s_totals_on_device[dev];
    return PIC_OK;
}

}  // namespace

extern "C" {

const char* pic_noalloc_last_error(void) { return t_error; }

int pic_cell_offsets_noalloc(int nx, int ny, int nz, double dx, double dy, double dz, double xmin, double ymin,
                             double zmin, long long n, const double* x, const double* y, const double* z,
                             unsigned int* offsets, void* cuda_stream) {
    t_error[0] = 0;
    if (nx < 1 || ny < 1 || nz < 1) return fail(PIC_EINVAL, "nx, ny, nz must be >= 1");
    const long long ncell = (long long)nx * ny * nz;
    if (ncell > PIC_NOALLOC_MAX_CELLS) {
        snprintf(t_error, sizeof t_error,
                 "pic_cell_offsets_noalloc: %lld cells exceed the built-in scratch (PIC_NOALLOC_MAX_CELLS = %lld); "
                 "use pic_sort + pic_get_cell_offsets with an arena instead", ncell, (long long)PIC_NOALLOC_MAX_CELLS);
        return PIC_EINVAL;
    }
    if (!(dx > 0.0) || !(dy > 0.0) || !(dz > 0.0) || !isfinite(dx) || !isfinite(dy) || !isfinite(dz) ||
        !isfinite(xmin) || !isfinite(ymin) || !isfinite(zmin))
        return fail(PIC_EINVAL, "dx, dy, dz must be positive and finite, xmin, ymin, zmin finite");
    if (n < 0 || n >= (1LL << 31)) return fail(PIC_EINVAL, "n must be in [0, 2^31)");
    if (!offsets) return fail(PIC_EINVAL, "offsets is NULL");
    if (n > 0 && (!x || !y || !z)) return fail(PIC_EINVAL, "x, y or z is NULL with n > 0");

    unsigned int* totals = nullptr;
    const int rc = scratch_on_current_device(&totals);
    if (rc != PIC_OK) return rc;

    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const long long nscan = ncell + 1;
    const int nchunks = (int)((nscan + CHUNK - 1) / CHUNK);   // <= PIC_NOALLOC_MAX_CHUNKS by the check above
    Box b{nx, ny, nz, xmin, ymin, zmin, 1.0 / dx, 1.0 / dy, 1.0 / dz};

    // The counters must start at zero: they are the caller's output buffer, cleared here.  The scratch needs no
    // clearing -- chunk_scan_kernel writes totals[0 .. nchunks) before anything reads them, and entries beyond
    // nchunks (left over from a larger earlier call) are never read.
    cudaError_t e = cudaMemsetAsync(offsets, 0, (size_t)nscan * sizeof(unsigned int), st);
    if (e != cudaSuccess) return fail(PIC_ECUDA, "cudaMemsetAsync(offsets)", e);
    if (n > 0) cell_count_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(b, x, y, z, n, offsets);
    chunk_scan_kernel<<<(unsigned)nchunks, CHUNK_T, 0, st>>>(offsets, nscan, totals);
    totals_scan_kernel<<<1, 1024, 0, st>>>(totals, nchunks);
    add_totals_kernel<<<(unsigned)nchunks, CHUNK_T, 0, st>>>(offsets, nscan, totals);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(PIC_ECUDA, "kernel launch", e);
    return PIC_OK;
}

}  // extern "C"
