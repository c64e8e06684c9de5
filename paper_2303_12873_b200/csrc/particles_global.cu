// particles_global.cu -- the order-independent particle path: one thread per
// particle, gather straight from the padded field arrays (L2/L1), Boris push,
// move, Esirkepov deposition with one global fp64 atomic (REDG.E.ADD.F64) per
// non-zero point, periodic wrap.  Correct for any particle order; it is what
// pic_step runs for a species that was never sorted, and what the fused tile
// kernel falls back to for a particle found outside its tile's halo.
// Also here: the rho diagnostic, the guard fold, the load validator, iota.
//
// Follows SURVEY 8(c.1) steps 1-5 (BASELINE.json:north_star parts 1-3;
// PAPER.md:45 "explicit ... iterate forward in time").
#include "particle_update.cuh"

namespace pic {

template <int N, int GV>
__global__ void __launch_bounds__(128) particles_global_kernel(Grid g, Fields f, Particles p, long long n, double q,
                                                               double h, DevStatus* status) {
    long long ip = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ip < n) update_particle_global<N, GV>(g, f, p, ip, q, h, status);
    if (ip == 0) atomicAdd(&status->n_global, (unsigned long long)n);
}

template <int GV>
static void launch_global_gv(const Grid& g, const Fields& f, const Particles& p, long long n, double q, double h,
                             int order, DevStatus* status, cudaStream_t st) {
    const int bs = 128;
    const unsigned nb = (unsigned)((n + bs - 1) / bs);
    if (order == 1) particles_global_kernel<1, GV><<<nb, bs, 0, st>>>(g, f, p, n, q, h, status);
    else if (order == 2) particles_global_kernel<2, GV><<<nb, bs, 0, st>>>(g, f, p, n, q, h, status);
    else particles_global_kernel<3, GV><<<nb, bs, 0, st>>>(g, f, p, n, q, h, status);
}

void launch_particles_global(const Grid& g, const Fields& f, const Particles& p, long long n, double q, double m,
                             int order, int gather_variant, DevStatus* status, cudaStream_t st) {
    if (n <= 0) return;
    const double h = q * g.dt / (2.0 * m);
    if (gather_variant) launch_global_gv<1>(g, f, p, n, q, h, order, status, st);
    else launch_global_gv<0>(g, f, p, n, q, h, order, status, st);
}

// ------------------------------------------------------------------- rho ----
template <int N>
__global__ void deposit_rho_kernel(Grid g, Particles p, long long n, double q, double* rho) {
    long long ip = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ip >= n) return;
    const double xi = (p.x[ip] - g.xmin) * g.inv_dx, et = (p.y[ip] - g.ymin) * g.inv_dy,
                 ze = (p.z[ip] - g.zmin) * g.inv_dz;
    double wx[N + 1], wy[N + 1], wz[N + 1];
    const int fx = shape_weights<N>(xi, wx), fy = shape_weights<N>(et, wy), fz = shape_weights<N>(ze, wz);
    const double qw = q * p.w[ip] * (g.inv_dx * g.inv_dy * g.inv_dz);
    double* base = rho + g.idx(fx, fy, fz);
#pragma unroll
    for (int c = 0; c <= N; ++c)
#pragma unroll
        for (int b = 0; b <= N; ++b)
#pragma unroll
            for (int a = 0; a <= N; ++a) atomicAdd(base + a + b * g.sy + c * g.sz, qw * wx[a] * wy[b] * wz[c]);
}

void launch_deposit_rho(const Grid& g, const Particles& p, long long n, double q, int order, double* rho,
                        cudaStream_t st) {
    if (n <= 0) return;
    const int bs = 128;
    const unsigned nb = (unsigned)((n + bs - 1) / bs);
    if (order == 1) deposit_rho_kernel<1><<<nb, bs, 0, st>>>(g, p, n, q, rho);
    else if (order == 2) deposit_rho_kernel<2><<<nb, bs, 0, st>>>(g, p, n, q, rho);
    else deposit_rho_kernel<3><<<nb, bs, 0, st>>>(g, p, n, q, rho);
}

// --------------------------------------------------------- guard fold ------
// interior[i,j,k] := sum over all periodic images of (i,j,k) inside the padded
// array (gather form: deterministic, no atomics).  Only cells within NG of a
// face have more than one image.
__device__ __forceinline__ int first_image(int i, int n) {   // smallest i + a*n >= -NG
    int a = (i + NG) / n;                                     // i + NG >= 0
    return i - a * n;
}

__global__ void fold_guards_kernel(Grid g, double* F) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    int j = blockIdx.y, k = blockIdx.z;
    if (i >= g.nx) return;
    const bool edge = i < NG || i >= g.nx - NG || j < NG || j >= g.ny - NG || k < NG || k >= g.nz - NG;
    if (!edge) return;
    double sum = 0.0;
    for (int kk = first_image(k, g.nz); kk < g.nz + NG; kk += g.nz)
        for (int jj = first_image(j, g.ny); jj < g.ny + NG; jj += g.ny)
            for (int ii = first_image(i, g.nx); ii < g.nx + NG; ii += g.nx) sum += F[g.idx(ii, jj, kk)];
    F[g.idx(i, j, k)] = sum;   // distinct threads own distinct interior cells; images are only read
}

// NOTE: the fold reads guard images while other threads overwrite interior
// cells; an interior cell is an image only of itself (|a| = 0), and it is read
// by its own thread only, so there is no race.
// the three J components in one launch (one thread per interior cell; only the edge cells do work)
__global__ void fold_guards3_kernel(Grid g, double* F0, double* F1, double* F2) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    int j = blockIdx.y, k = blockIdx.z;
    if (i >= g.nx) return;
    const bool edge = i < NG || i >= g.nx - NG || j < NG || j >= g.ny - NG || k < NG || k >= g.nz - NG;
    if (!edge) return;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    for (int kk = first_image(k, g.nz); kk < g.nz + NG; kk += g.nz)
        for (int jj = first_image(j, g.ny); jj < g.ny + NG; jj += g.ny)
            for (int ii = first_image(i, g.nx); ii < g.nx + NG; ii += g.nx) {
                const long long o = g.idx(ii, jj, kk);
                s0 += F0[o];
                s1 += F1[o];
                s2 += F2[o];
            }
    const long long o = g.idx(i, j, k);
    F0[o] = s0;
    F1[o] = s1;
    F2[o] = s2;
}

void launch_fold_guards3(const Grid& g, double* F0, double* F1, double* F2, cudaStream_t st) {
    dim3 bs(128, 1, 1), nb((g.nx + 127) / 128, g.ny, g.nz);
    fold_guards3_kernel<<<nb, bs, 0, st>>>(g, F0, F1, F2);
}

void launch_fold_guards(const Grid& g, double* F, cudaStream_t st) {
    dim3 bs(128, 1, 1), nb((g.nx + 127) / 128, g.ny, g.nz);
    fold_guards_kernel<<<nb, bs, 0, st>>>(g, F);
}

// ------------------------------------------------------- load validator ----
__global__ void validate_kernel(Grid g, Particles p, long long n, DevStatus* status) {
    long long ip = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ip >= n) return;
    const double x = p.x[ip], y = p.y[ip], z = p.z[ip];
    bool ok = x >= g.xmin && x < g.xmax && y >= g.ymin && y < g.ymax && z >= g.zmin && z < g.zmax;
    ok = ok && isfinite(p.ux[ip]) && isfinite(p.uy[ip]) && isfinite(p.uz[ip]) && isfinite(p.w[ip]);
    if (!ok) status->ebox = 1;
}

void launch_validate(const Grid& g, const Particles& p, long long n, DevStatus* status, cudaStream_t st) {
    if (n <= 0) return;
    validate_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(g, p, n, status);
}

__global__ void iota_kernel(unsigned long long* id, long long n) {
    long long ip = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ip < n) id[ip] = (unsigned long long)ip;
}

void launch_iota(unsigned long long* id, long long n, cudaStream_t st) {
    if (n <= 0) return;
    iota_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(id, n);
}

}  // namespace pic
