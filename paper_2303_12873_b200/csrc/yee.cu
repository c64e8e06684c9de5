// yee.cu -- Yee FDTD update of B (half step) and E (full step) on the padded
// staggered grid (BASELINE.json:north_star part 4).
//
//   Bx -= dth[(Ez[i,j+1,k]-Ez)/dy - (Ey[i,j,k+1]-Ey)/dz]   (forward differences)
//   Ex += dt [c^2((Bz-Bz[i,j-1,k])/dy - (By-By[i,j,k-1])/dz) - Jx/eps0]  (backward)
//   and cyclic permutations.
//
// Each thread owns one interior cell, computes the three components there and
// stores the result to the interior location AND to every periodic guard
// image of that cell, so no separate guard-exchange pass is needed: after a
// push the updated component is valid on the whole padded array.
// HBM-bound: 72 B/cell (B push), 96 B/cell (E push) algorithmic.
//
// Two implementations of each push:
//   *_kernel      one thread per cell, every operand a global load (12 loads per cell; the +-1 rows in
//                 y and z miss L1, so the kernel is L1/L2-throughput bound at ~40 % of the HBM roofline);
//   *_tma_kernel  one block per 32 x 8 x 4 (B push) or 32 x 8 x 8 (E push) tile: the three curl operands (+ a one-cell halo) are staged
//                 in shared memory by TMA (cp.async.bulk.tensor.3d, one thread, mbarrier
//                 completion) while the threads fetch the component they update; the padded guard cells
//                 mean a box never wraps, and boxes that poke out of the array are zero-filled.
#include <cuda.h>

#include <algorithm>

#include "pic_internal.h"

namespace pic {

__device__ __forceinline__ int first_img(int i, int n) {   // smallest i + a*n >= -NG
    return i - ((i + NG) / n) * n;
}

__device__ __forceinline__ bool is_edge(const Grid& g, int i, int j, int k) {
    return i < NG || i >= g.nx - NG || j < NG || j >= g.ny - NG || k < NG || k >= g.nz - NG;
}

// store v0,v1,v2 of three components at every periodic image of (i,j,k) except itself
__device__ __noinline__ void store_images3(const Grid& g, double* F0, double* F1, double* F2, int i, int j, int k,
                                           double v0, double v1, double v2) {
    for (int kk = first_img(k, g.nz); kk < g.nz + NG; kk += g.nz)
        for (int jj = first_img(j, g.ny); jj < g.ny + NG; jj += g.ny)
            for (int ii = first_img(i, g.nx); ii < g.nx + NG; ii += g.nx) {
                if (ii == i && jj == j && kk == k) continue;
                const long long o = g.idx(ii, jj, kk);
                F0[o] = v0;
                F1[o] = v1;
                F2[o] = v2;
            }
}

__global__ void __launch_bounds__(128) push_B_kernel(Grid g, Fields f, double cdx, double cdy, double cdz) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    if (i >= g.nx) return;
    const long long o = g.idx(i, j, k);
    const double ex = f.Ex[o], ey = f.Ey[o], ez = f.Ez[o];
    const double bx = f.Bx[o] - (cdy * (f.Ez[o + g.sy] - ez) - cdz * (f.Ey[o + g.sz] - ey));
    const double by = f.By[o] - (cdz * (f.Ex[o + g.sz] - ex) - cdx * (f.Ez[o + 1] - ez));
    const double bz = f.Bz[o] - (cdx * (f.Ey[o + 1] - ey) - cdy * (f.Ex[o + g.sy] - ex));
    f.Bx[o] = bx;
    f.By[o] = by;
    f.Bz[o] = bz;
    if (is_edge(g, i, j, k)) store_images3(g, f.Bx, f.By, f.Bz, i, j, k, bx, by, bz);
}

__global__ void __launch_bounds__(128) push_E_kernel(Grid g, Fields f, double cdx, double cdy, double cdz,
                                                     double dt_eps0) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    if (i >= g.nx) return;
    const long long o = g.idx(i, j, k);
    const double bx = f.Bx[o], by = f.By[o], bz = f.Bz[o];
    const double ex = f.Ex[o] + (cdy * (bz - f.Bz[o - g.sy]) - cdz * (by - f.By[o - g.sz])) - dt_eps0 * f.Jx[o];
    const double ey = f.Ey[o] + (cdz * (bx - f.Bx[o - g.sz]) - cdx * (bz - f.Bz[o - 1])) - dt_eps0 * f.Jy[o];
    const double ez = f.Ez[o] + (cdx * (by - f.By[o - 1]) - cdy * (bx - f.Bx[o - g.sy])) - dt_eps0 * f.Jz[o];
    f.Ex[o] = ex;
    f.Ey[o] = ey;
    f.Ez[o] = ez;
    if (is_edge(g, i, j, k)) store_images3(g, f.Ex, f.Ey, f.Ez, i, j, k, ex, ey, ez);
}

// ---- TMA-staged variant ------------------------------------------------------------------------
namespace {

constexpr int YTX = 32, YTY = 8;                           // cells per block in x, y (one thread each)
constexpr int YTZ_B = 4, YTZ_E = 8;                        // z planes a thread walks (measured best at 256^3: profiles/r02_yee.md)                  // cells per block
// Staged box: the tile plus one halo cell in y and z and, in x, 2 cells: with 8-byte elements the box corner
// must sit on an EVEN x coordinate (TMA wants the first byte of a box row 16-byte aligned; an odd coordinate
// raises "illegal instruction"), so the E push (backward differences) starts 2 cells below the tile, not 1.
// Row = 34 or 36 doubles = 272 / 288 B: a multiple of 16 B as TMA requires.
constexpr int YBY = YTY + 1;
template <int HX, int TZ> struct YeeBox {
    static constexpr int BX = YTX + HX, BZ = TZ + 1;
    static constexpr int SZ = BX * YBY * BZ;
    static constexpr int PAD = (SZ + 15) / 16 * 16;        // every TMA destination starts on a 128-byte boundary
};
constexpr int YNT = 256;

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned phase) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(phase) : "memory");
}
// one 3-D box of a padded component -> shared memory; (x, y, z) = padded element coordinates of its corner
__device__ __forceinline__ void tma_load_box(double* dst, const CUtensorMap* map, unsigned long long* bar, int x,
                                             int y, int z) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(smem_u32(dst)), "l"(reinterpret_cast<unsigned long long>(map)), "r"(x), "r"(y), "r"(z),
        "r"(smem_u32(bar)) : "memory");
}

template <int HX, int TZ> struct YeeSmem {
    alignas(128) double box[3][YeeBox<HX, TZ>::PAD];
    alignas(8) unsigned long long bar;
};

// Box corner = (tile's first cell) - (shx, sh, sh): sh = 0 for forward differences (B push), 1 for backward
// differences (E push, shx = 2 to stay on an even x coordinate).
template <int HX, int TZ>
__device__ __forceinline__ void stage_boxes(YeeSmem<HX, TZ>& sm, const CUtensorMap* m0, const CUtensorMap* m1,
                                            const CUtensorMap* m2, int t0x, int t0y, int t0z, int shx, int sh) {
    if (threadIdx.x == 0) mbar_init(&sm.bar, 1);
    __syncthreads();
    if (threadIdx.x == 0) {
        mbar_expect_tx(&sm.bar, 3u * YeeBox<HX, TZ>::SZ * (unsigned)sizeof(double));
        tma_load_box(sm.box[0], m0, &sm.bar, t0x + NG - shx, t0y + NG - sh, t0z + NG - sh);
        tma_load_box(sm.box[1], m1, &sm.bar, t0x + NG - shx, t0y + NG - sh, t0z + NG - sh);
        tma_load_box(sm.box[2], m2, &sm.bar, t0x + NG - shx, t0y + NG - sh, t0z + NG - sh);
    }
}

}  // namespace

template <int YTZ>
__global__ void __launch_bounds__(YNT) push_B_tma_kernel(Grid g, Fields f, double cdx, double cdy, double cdz,
                                                         const __grid_constant__ CUtensorMap mEx,
                                                         const __grid_constant__ CUtensorMap mEy,
                                                         const __grid_constant__ CUtensorMap mEz) {
    extern __shared__ __align__(128) unsigned char yee_smem_raw[];
    constexpr int YBX = YeeBox<2, YTZ>::BX;
    YeeSmem<2, YTZ>& sm = *reinterpret_cast<YeeSmem<2, YTZ>*>(yee_smem_raw);
    const int t0x = blockIdx.x * YTX, t0y = blockIdx.y * YTY, t0z = blockIdx.z * YTZ;
    stage_boxes<2, YTZ>(sm, &mEx, &mEy, &mEz, t0x, t0y, t0z, 0, 0);
    const int tx = threadIdx.x % YTX, ty = threadIdx.x / YTX;     // 32 x 8 threads, each walks the 8 z planes
    const int i = t0x + tx, j = t0y + ty;
    const bool in_xy = i < g.nx && j < g.ny;
    double bx[YTZ], by[YTZ], bz[YTZ];
#pragma unroll
    for (int c = 0; c < YTZ; ++c) {
        const bool ok = in_xy && t0z + c < g.nz;
        const long long o = g.idx(i, j, t0z + c);
        bx[c] = ok ? f.Bx[o] : 0.0;
        by[c] = ok ? f.By[o] : 0.0;
        bz[c] = ok ? f.Bz[o] : 0.0;
    }
    mbar_wait(&sm.bar, 0);
    const double* Ex = sm.box[0] + tx + YBX * ty;
    const double* Ey = sm.box[1] + tx + YBX * ty;
    const double* Ez = sm.box[2] + tx + YBX * ty;
#pragma unroll
    for (int c = 0; c < YTZ; ++c) {
        const int k = t0z + c;
        if (!(in_xy && k < g.nz)) continue;
        const int w = YBX * YBY * c;
        const double ex = Ex[w], ey = Ey[w], ez = Ez[w];
        const double nbx = bx[c] - (cdy * (Ez[w + YBX] - ez) - cdz * (Ey[w + YBX * YBY] - ey));
        const double nby = by[c] - (cdz * (Ex[w + YBX * YBY] - ex) - cdx * (Ez[w + 1] - ez));
        const double nbz = bz[c] - (cdx * (Ey[w + 1] - ey) - cdy * (Ex[w + YBX] - ex));
        const long long o = g.idx(i, j, k);
        f.Bx[o] = nbx;
        f.By[o] = nby;
        f.Bz[o] = nbz;
        if (is_edge(g, i, j, k)) store_images3(g, f.Bx, f.By, f.Bz, i, j, k, nbx, nby, nbz);
    }
}

template <int YTZ>
__global__ void __launch_bounds__(YNT) push_E_tma_kernel(Grid g, Fields f, double cdx, double cdy, double cdz,
                                                         double dt_eps0, const __grid_constant__ CUtensorMap mBx,
                                                         const __grid_constant__ CUtensorMap mBy,
                                                         const __grid_constant__ CUtensorMap mBz) {
    extern __shared__ __align__(128) unsigned char yee_smem_raw[];
    constexpr int YBX = YeeBox<4, YTZ>::BX;
    YeeSmem<4, YTZ>& sm = *reinterpret_cast<YeeSmem<4, YTZ>*>(yee_smem_raw);
    const int t0x = blockIdx.x * YTX, t0y = blockIdx.y * YTY, t0z = blockIdx.z * YTZ;
    stage_boxes<4, YTZ>(sm, &mBx, &mBy, &mBz, t0x, t0y, t0z, 2, 1);
    const int tx = threadIdx.x % YTX, ty = threadIdx.x / YTX;
    const int i = t0x + tx, j = t0y + ty;
    const bool in_xy = i < g.nx && j < g.ny;
    double ex[YTZ], ey[YTZ], ez[YTZ], jx[YTZ], jy[YTZ], jz[YTZ];     // in flight while the TMA boxes land
#pragma unroll
    for (int c = 0; c < YTZ; ++c) {
        const bool ok = in_xy && t0z + c < g.nz;
        const long long o = g.idx(i, j, t0z + c);
        ex[c] = ok ? f.Ex[o] : 0.0;
        ey[c] = ok ? f.Ey[o] : 0.0;
        ez[c] = ok ? f.Ez[o] : 0.0;
        jx[c] = ok ? f.Jx[o] : 0.0;
        jy[c] = ok ? f.Jy[o] : 0.0;
        jz[c] = ok ? f.Jz[o] : 0.0;
    }
    mbar_wait(&sm.bar, 0);
    const double* Bx = sm.box[0] + (tx + 2) + YBX * (ty + 1) + YBX * YBY;
    const double* By = sm.box[1] + (tx + 2) + YBX * (ty + 1) + YBX * YBY;
    const double* Bz = sm.box[2] + (tx + 2) + YBX * (ty + 1) + YBX * YBY;
#pragma unroll
    for (int c = 0; c < YTZ; ++c) {
        const int k = t0z + c;
        if (!(in_xy && k < g.nz)) continue;
        const int w = YBX * YBY * c;
        const double bx = Bx[w], by = By[w], bz = Bz[w];
        const long long o = g.idx(i, j, k);
        // same operation order as the plain kernel: (E + curl term) - dt/eps0 J
        const double nex = (ex[c] + (cdy * (bz - Bz[w - YBX]) - cdz * (by - By[w - YBX * YBY]))) - dt_eps0 * jx[c];
        const double ney = (ey[c] + (cdz * (bx - Bx[w - YBX * YBY]) - cdx * (bz - Bz[w - 1]))) - dt_eps0 * jy[c];
        const double nez = (ez[c] + (cdx * (by - By[w - 1]) - cdy * (bx - Bx[w - YBX]))) - dt_eps0 * jz[c];
        f.Ex[o] = nex;
        f.Ey[o] = ney;
        f.Ez[o] = nez;
        if (is_edge(g, i, j, k)) store_images3(g, f.Ex, f.Ey, f.Ez, i, j, k, nex, ney, nez);
    }
}

// (A persistent variant -- one block per SM streaming items through a TMA ring -- was measured in round 2 at 2.0 TB/s
// against 4.7 TB/s for one tile per block and removed in round 3; the measurement stays in profiles/r02_yee.md.)

void launch_push_B(const Grid& g, const Fields& f, double dth, const YeeMaps* maps, cudaStream_t st) {
    const double cdx = dth * g.inv_dx, cdy = dth * g.inv_dy, cdz = dth * g.inv_dz;
    if (maps && maps->valid) {
        dim3 nb((g.nx + YTX - 1) / YTX, (g.ny + YTY - 1) / YTY, (g.nz + YTZ_B - 1) / YTZ_B);
        const CUtensorMap* m = reinterpret_cast<const CUtensorMap*>(maps->map);
        push_B_tma_kernel<YTZ_B><<<nb, YNT, sizeof(YeeSmem<2, YTZ_B>), st>>>(g, f, cdx, cdy, cdz, m[0], m[1], m[2]);
    } else {
        dim3 bs(128, 1, 1), nb((g.nx + 127) / 128, g.ny, g.nz);
        push_B_kernel<<<nb, bs, 0, st>>>(g, f, cdx, cdy, cdz);
    }
}

void launch_push_E(const Grid& g, const Fields& f, double dt, const YeeMaps* maps, cudaStream_t st) {
    const double c2dt = C_LIGHT * C_LIGHT * dt;
    const double cdx = c2dt * g.inv_dx, cdy = c2dt * g.inv_dy, cdz = c2dt * g.inv_dz;
    if (maps && maps->valid) {
        dim3 nb((g.nx + YTX - 1) / YTX, (g.ny + YTY - 1) / YTY, (g.nz + YTZ_E - 1) / YTZ_E);
        const CUtensorMap* m = reinterpret_cast<const CUtensorMap*>(maps->map);
        push_E_tma_kernel<YTZ_E><<<nb, YNT, sizeof(YeeSmem<4, YTZ_E>), st>>>(g, f, cdx, cdy, cdz, dt / EPS0, m[3], m[4], m[5]);
    } else {
        dim3 bs(128, 1, 1), nb((g.nx + 127) / 128, g.ny, g.nz);
        push_E_kernel<<<nb, bs, 0, st>>>(g, f, cdx, cdy, cdz, dt / EPS0);
    }
}

// Tensor maps of the six padded E,B components (rank 3, fp64, no swizzle, zero fill outside the array),
// box = (YTX + 2) x YBY x (YTZ_B + 1) for E (read by the B push), (YTX + 4) x YBY x (YTZ_E + 1) for B.  The driver entry point is fetched through the runtime (no link-time libcuda).
int make_yee_maps(const Grid& g, const Fields& f, YeeMaps* out) {
    static_assert(sizeof(CUtensorMap) == 128 && sizeof(out->map) == 6 * 128, "YeeMaps storage");
    out->valid = 0;
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                 const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                 CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return 1;
    }
    double* comp[6] = {f.Ex, f.Ey, f.Ez, f.Bx, f.By, f.Bz};
    CUtensorMap* m = reinterpret_cast<CUtensorMap*>(out->map);
    const cuuint64_t dims[3] = {(cuuint64_t)g.px, (cuuint64_t)g.py, (cuuint64_t)g.pz};
    const cuuint64_t strides[2] = {(cuuint64_t)g.px * 8, (cuuint64_t)g.px * (cuuint64_t)g.py * 8};
    const cuuint32_t estr[3] = {1, 1, 1};
    for (int k = 0; k < 6; ++k) {
        const cuuint32_t box[3] = {(cuuint32_t)(k < 3 ? YeeBox<2, YTZ_B>::BX : YeeBox<4, YTZ_E>::BX), YBY,
                                   (cuuint32_t)(k < 3 ? YeeBox<2, YTZ_B>::BZ : YeeBox<4, YTZ_E>::BZ)};
        CUresult r = ((EncodeFn)fn)(&m[k], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, comp[k], dims, strides, box, estr,
                                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                    CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return 2;
    }
    if (cudaFuncSetAttribute(push_B_tma_kernel<YTZ_B>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)sizeof(YeeSmem<2, YTZ_B>)) !=
            cudaSuccess ||
        cudaFuncSetAttribute(push_E_tma_kernel<YTZ_E>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)sizeof(YeeSmem<4, YTZ_E>)) !=
            cudaSuccess) {
        cudaGetLastError();
        return 3;
    }
    out->valid = 1;
    return 0;
}


// Periodic images of one component from its interior (used after pic_set_fields).
__global__ void fill_guards_kernel(Grid g, double* F) {
    const int ii = (int)(blockIdx.x * blockDim.x + threadIdx.x) - NG;
    const int jj = (int)blockIdx.y - NG, kk = (int)blockIdx.z - NG;
    if (ii >= g.nx + NG) return;
    if (ii >= 0 && ii < g.nx && jj >= 0 && jj < g.ny && kk >= 0 && kk < g.nz) return;
    const int i = ((ii % g.nx) + g.nx) % g.nx, j = ((jj % g.ny) + g.ny) % g.ny, k = ((kk % g.nz) + g.nz) % g.nz;
    F[g.idx(ii, jj, kk)] = F[g.idx(i, j, k)];
}

void launch_fill_guards(const Grid& g, double* F, cudaStream_t st) {
    dim3 bs(128, 1, 1), nb((g.nx + 2 * NG + 127) / 128, g.ny + 2 * NG, g.nz + 2 * NG);
    fill_guards_kernel<<<nb, bs, 0, st>>>(g, F);
}

// ---- binomial smoothing of one component (pic_set_option "smooth_passes") -------------
// One pass = the 1-2-1 filter along x, then y, then z, periodic.  The kernel reads the component with its
// periodic guard images filled and evaluates the three filters in that order on the 3 x 3 x 3 neighbourhood of
// its cell (the same operations, in the same order, as three sweeps over the whole array), writing the
// interior of `out`.
__global__ void smooth121_kernel(Grid g, const double* __restrict__ F, double* __restrict__ out) {
    const int i = (int)(blockIdx.x * blockDim.x + threadIdx.x), j = (int)blockIdx.y, k = (int)blockIdx.z;
    if (i >= g.nx) return;
    const double* c = F + g.idx(i, j, k);
    double tz[3];
#pragma unroll
    for (int dz = -1; dz <= 1; ++dz) {
        double ty[3];
#pragma unroll
        for (int dy = -1; dy <= 1; ++dy) {
            const double* r = c + g.sy * dy + g.sz * dz;
            ty[dy + 1] = 0.25 * r[-1] + 0.5 * r[0] + 0.25 * r[1];
        }
        tz[dz + 1] = 0.25 * ty[0] + 0.5 * ty[1] + 0.25 * ty[2];
    }
    out[g.idx(i, j, k)] = 0.25 * tz[0] + 0.5 * tz[1] + 0.25 * tz[2];
}

__global__ void copy_interior_kernel(Grid g, const double* __restrict__ src, double* __restrict__ dst) {
    const int i = (int)(blockIdx.x * blockDim.x + threadIdx.x), j = (int)blockIdx.y, k = (int)blockIdx.z;
    if (i < g.nx) dst[g.idx(i, j, k)] = src[g.idx(i, j, k)];
}

// F := `npass` binomial passes of F (interior; the guard cells of F are left as periodic images of the last
// but one pass and must not be relied on).  tmp = one padded scratch component.  Returns kernels launched.
int launch_smooth_binomial(const Grid& g, double* F, double* tmp, int npass, cudaStream_t st) {
    dim3 bs(128, 1, 1), nb((g.nx + 127) / 128, g.ny, g.nz);
    int launches = 0;
    for (int p = 0; p < npass; ++p) {
        launch_fill_guards(g, F, st);
        smooth121_kernel<<<nb, bs, 0, st>>>(g, F, tmp);
        copy_interior_kernel<<<nb, bs, 0, st>>>(g, tmp, F);
        launches += 3;
    }
    return launches;
}

}  // namespace pic
