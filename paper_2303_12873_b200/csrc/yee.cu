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

void launch_push_B(const Grid& g, const Fields& f, double dth, bool /*tma*/, cudaStream_t st) {
    dim3 bs(128, 1, 1), nb((g.nx + 127) / 128, g.ny, g.nz);
    push_B_kernel<<<nb, bs, 0, st>>>(g, f, dth * g.inv_dx, dth * g.inv_dy, dth * g.inv_dz);
}

void launch_push_E(const Grid& g, const Fields& f, double dt, bool /*tma*/, cudaStream_t st) {
    dim3 bs(128, 1, 1), nb((g.nx + 127) / 128, g.ny, g.nz);
    const double c2dt = C_LIGHT * C_LIGHT * dt;
    push_E_kernel<<<nb, bs, 0, st>>>(g, f, c2dt * g.inv_dx, c2dt * g.inv_dy, c2dt * g.inv_dz, dt / EPS0);
}

int yee_num_launches(bool) { return 1; }

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

}  // namespace pic
