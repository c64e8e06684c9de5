// peaks.cu -- micro-probes of the machine rates the rooflines of bench.py and
// DESIGN.md section 5 are quoted against ("Builder must measure
// first: fp64 FMA peak ..., shared-memory LDS.64 wavefront rate with 1/2/4
// distinct addresses per warp ..., global fp64 red.add rate at L2").  They
// sit behind a C ABI of their own (include/pic_probes.h, libpic_probes.so) so that one committed
// command -- python -m paper_2303_12873_b200.peaks -- prints the table and
// the same command can be put under ncu for the wavefront counters.
// Unlike the simulation calls, the probes allocate their few MB of scratch
// themselves (cudaMalloc on the current device, default stream) and free it:
// they are built into a separate library so that libpic_b200.so never allocates.
#include <stdio.h>

#include "pic_internal.h"
#include "../../include/pic_probes.h"

namespace pic {
namespace {

// ---- fp64 pipe: DFMA issue rate ---------------------------------------------------------------
__global__ void probe_dfma_kernel(int iters, long long* clk, double* sink) {
    double a[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) a[k] = 1.0 + 1e-9 * (threadIdx.x + k);
    const double m = 1.0000001, c = 1e-7;
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] = fma(a[k], m, c);      // 8 independent chains, 32 DFMA per trip
    }
    const long long t1 = clock64();
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += a[k];
    if (s == 12345.678) sink[0] = s;
    if (threadIdx.x == 0) clk[blockIdx.x] = t1 - t0;
}

// ---- fp64 tensor path: DMMA m8n8k4 (256 FMA per warp instruction) ----------------------------------
__global__ void probe_dmma_kernel(int iters, long long* clk, double* sink) {
    double c[8][2];
#pragma unroll
    for (int k = 0; k < 8; ++k) { c[k][0] = 1e-9 * threadIdx.x; c[k][1] = 1e-9 * k; }
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-7;
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k)      // 8 independent accumulator fragments
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                         : "+d"(c[k][0]), "+d"(c[k][1]) : "d"(a), "d"(b));
    }
    const long long t1 = clock64();
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += c[k][0] + c[k][1];
    if (s == 12345.678) sink[0] = s;
    if (threadIdx.x == 0) clk[blockIdx.x] = t1 - t0;
}

// ---- shared-memory return path: LDS.64 / LDS.128 with a given lane -> word map -------------------
// Every active lane of every warp reads word lane_word[lane] (+ a per-load offset that keeps the
// bank pattern) of a shared array laid out like the tile kernel's stencil; eight independent loads
// per trip.  Lanes outside `active` leave before the loop, so the warp's loads carry fewer lanes.
constexpr int PROBE_SMEM_WORDS = 6144;
template <int VEC>
__global__ void probe_lds_kernel(const int* __restrict__ lane_word, unsigned active, int plane_words, int iters,
                                 int zero, long long* clk, double* sink) {
    __shared__ __align__(16) double sm[PROBE_SMEM_WORDS];
    for (int i = threadIdx.x; i < PROBE_SMEM_WORDS; i += blockDim.x) sm[i] = 0.5 * i;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    if (!((active >> lane) & 1u)) return;
    const double* base = sm + lane_word[lane];
    double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
        // `zero` is 0 at run time but opaque to the compiler: the addresses change with the trip as far as it
        // can tell, so the eight loads are issued on every trip (with trip-invariant addresses the whole
        // loop collapsed into one trip, volatile asm or not).
        const double* a = base + it * zero;
        double v[8], w[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {       // plain loads: ptxas may keep all eight in flight
            if constexpr (VEC == 8) {
                v[k] = a[k * plane_words];
                w[k] = 0.0;
            } else {
                const double2 t = *reinterpret_cast<const double2*>(a + k * plane_words);
                v[k] = t.x;
                w[k] = t.y;
            }
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            acc[k] += v[k];
            if constexpr (VEC == 16) acc[k] += w[k];
        }
    }
    const long long t1 = clock64();
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += acc[k];
    if (s == 12345.678) sink[0] = s;
    if (threadIdx.x == __ffs(active) - 1) clk[blockIdx.x] = t1 - t0;
}

// ---- L2 atomics: red.global.add.f64 ------------------------------------------------------------
// pattern 0: the 32 lanes of a warp add to 32 consecutive doubles (8 sectors of 32 B per instruction)
//         1: every lane its own sector (stride 4 doubles: 32 sectors per instruction)
//         2: every lane its own 128-byte line (stride 16 doubles)
//         3: all 32 lanes the same double (one sector, 32-way contention)
//         4: flush-like: lane = (cell-group g = lane >> 2, plane s = lane & 3): 8 unrelated places x 4 planes
//            `plane` doubles apart (what an unmerged per-cell accumulator flush issues)
//         5: as 4 but the 4 lanes of a group on 4 consecutive doubles (x-adjacent nodes)
// Successive REDs of a thread jump through the footprint (span_mask + 1 = the largest power of two that
// leaves room for the pattern), so that the working set is about `footprint` doubles.
__global__ void probe_red_kernel(double* J, unsigned long long span_mask, int pattern, long long plane, int n_per_thread) {
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    unsigned long long h = (unsigned long long)warp * 0x9E3779B97F4A7C15ull + 0x1234567ull;
    for (int it = 0; it < n_per_thread; ++it) {
        h = h * 6364136223846793005ull + 1442695040888963407ull;
        const long long base = (long long)((h >> 20) & span_mask & ~3ull);      // sector-aligned start inside the footprint
        long long o;
        if (pattern == 0) o = base + lane;
        else if (pattern == 1) o = base + 4 * lane;
        else if (pattern == 2) o = base + 16 * lane;
        else if (pattern == 3) o = base;
        else {
            const int g = lane >> 2, s = lane & 3;
            unsigned long long hg = (h ^ ((unsigned long long)g * 0xD6E8FEB86659FD93ull)) * 0x9E3779B97F4A7C15ull;
            const long long bg = (long long)((hg >> 20) & span_mask & ~3ull);
            o = (pattern == 4) ? bg + plane * s : bg + s;
        }
        asm volatile("red.global.add.f64 [%0], %1;" ::"l"(J + o), "d"(1.0) : "memory");
    }
}

int sm_count() {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
    return n;
}

// median of the per-block cycle counts (one block per SM)
double median_clk(long long* d_clk, int n) {
    long long* h = new long long[n];
    cudaMemcpy(h, d_clk, sizeof(long long) * n, cudaMemcpyDeviceToHost);
    for (int i = 1; i < n; ++i) {
        long long v = h[i];
        int j = i - 1;
        while (j >= 0 && h[j] > v) { h[j + 1] = h[j]; --j; }
        h[j + 1] = v;
    }
    const double m = (double)h[n / 2];
    delete[] h;
    return m;
}

}  // namespace
}  // namespace pic

using namespace pic;

extern "C" {

int pic_probe_dfma(int warps_per_sm, int iters, double* clk_per_warp_instr) {
    if (!clk_per_warp_instr || warps_per_sm < 1 || warps_per_sm > 32 || iters < 1) return PIC_EINVAL;
    const int nsm = sm_count();
    if (nsm <= 0) return PIC_ECUDA;
    long long* clk = nullptr;
    double* sink = nullptr;
    if (cudaMalloc(&clk, sizeof(long long) * nsm) != cudaSuccess || cudaMalloc(&sink, 8) != cudaSuccess) return PIC_ENOMEM;
    probe_dfma_kernel<<<nsm, 32 * warps_per_sm>>>(iters, clk, sink);
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) *clk_per_warp_instr = median_clk(clk, nsm) / ((double)iters * 32.0 * warps_per_sm);
    cudaFree(clk);
    cudaFree(sink);
    return e == cudaSuccess ? PIC_OK : PIC_ECUDA;
}

int pic_probe_dmma(int warps_per_sm, int iters, double* clk_per_warp_instr) {
    if (!clk_per_warp_instr || warps_per_sm < 1 || warps_per_sm > 32 || iters < 1) return PIC_EINVAL;
    const int nsm = sm_count();
    if (nsm <= 0) return PIC_ECUDA;
    long long* clk = nullptr;
    double* sink = nullptr;
    if (cudaMalloc(&clk, sizeof(long long) * nsm) != cudaSuccess || cudaMalloc(&sink, 8) != cudaSuccess) return PIC_ENOMEM;
    probe_dmma_kernel<<<nsm, 32 * warps_per_sm>>>(iters, clk, sink);
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) *clk_per_warp_instr = median_clk(clk, nsm) / ((double)iters * 8.0 * warps_per_sm);
    cudaFree(clk);
    cudaFree(sink);
    return e == cudaSuccess ? PIC_OK : PIC_ECUDA;
}

int pic_probe_lds(int vec_bytes, const int* lane_word, unsigned int active_mask, int plane_words, int warps_per_sm,
                  int iters, double* clk_per_warp_instr) {
    if (!clk_per_warp_instr || !lane_word || (vec_bytes != 8 && vec_bytes != 16) || !active_mask || warps_per_sm < 1 ||
        warps_per_sm > 32 || iters < 1 || plane_words < 0)
        return PIC_EINVAL;
    for (int l = 0; l < 32; ++l)
        if (lane_word[l] < 0 || lane_word[l] + 7 * plane_words + 2 > PROBE_SMEM_WORDS ||
            (vec_bytes == 16 && (lane_word[l] & 1)))
            return PIC_EINVAL;
    if (vec_bytes == 16 && (plane_words & 1)) return PIC_EINVAL;
    const int nsm = sm_count();
    if (nsm <= 0) return PIC_ECUDA;
    long long* clk = nullptr;
    double* sink = nullptr;
    int* dw = nullptr;
    if (cudaMalloc(&clk, sizeof(long long) * nsm) != cudaSuccess || cudaMalloc(&sink, 8) != cudaSuccess ||
        cudaMalloc(&dw, 128) != cudaSuccess)
        return PIC_ENOMEM;
    cudaMemcpy(dw, lane_word, 128, cudaMemcpyHostToDevice);
    if (vec_bytes == 8) probe_lds_kernel<8><<<nsm, 32 * warps_per_sm>>>(dw, active_mask, plane_words, iters, 0, clk, sink);
    else probe_lds_kernel<16><<<nsm, 32 * warps_per_sm>>>(dw, active_mask, plane_words, iters, 0, clk, sink);
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) *clk_per_warp_instr = median_clk(clk, nsm) / ((double)iters * 8.0 * warps_per_sm);
    cudaFree(clk);
    cudaFree(sink);
    cudaFree(dw);
    return e == cudaSuccess ? PIC_OK : PIC_ECUDA;
}

int pic_probe_red(int pattern, long long footprint_doubles, long long plane_doubles, int reds_per_thread,
                  double* lane_reds_per_s) {
    if (!lane_reds_per_s || pattern < 0 || pattern > 5 || reds_per_thread < 1 || plane_doubles < 1 ||
        footprint_doubles < 8 * plane_doubles + 4096)
        return PIC_EINVAL;
    const int nsm = sm_count();
    if (nsm <= 0) return PIC_ECUDA;
    double* J = nullptr;
    if (cudaMalloc(&J, sizeof(double) * (size_t)footprint_doubles) != cudaSuccess) return PIC_ENOMEM;
    cudaMemset(J, 0, sizeof(double) * (size_t)footprint_doubles);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int nb = nsm * 8, nt = 256;
    unsigned long long span = 1;
    while (2 * span <= (unsigned long long)(footprint_doubles - 4 * plane_doubles - 1024)) span *= 2;
    probe_red_kernel<<<nb, nt>>>(J, span - 1, pattern, plane_doubles, reds_per_thread / 4 + 1);   // warm-up
    cudaEventRecord(e0);
    probe_red_kernel<<<nb, nt>>>(J, span - 1, pattern, plane_doubles, reds_per_thread);
    cudaEventRecord(e1);
    cudaError_t e = cudaDeviceSynchronize();
    float ms = 0.f;
    if (e == cudaSuccess) {
        cudaEventElapsedTime(&ms, e0, e1);
        *lane_reds_per_s = (double)nb * nt * (double)reds_per_thread / (1e-3 * ms);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(J);
    return e == cudaSuccess ? PIC_OK : PIC_ECUDA;
}

}  // extern "C"
