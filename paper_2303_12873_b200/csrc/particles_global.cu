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

template <int N, int GV, int DV, class T>
__global__ void __launch_bounds__(128) particles_global_kernel(Grid g, Fields f, Particles p, long long n, double q,
                                                               double h, DevStatus* status) {
    long long ip = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ip < n) update_particle_global<N, GV, DV, T>(g, f, p, ip, q, h, status);
    if (ip == 0) atomicAdd(&status->n_global, (unsigned long long)n);
}

template <int GV, int DV, class T>
static void launch_global_gv(const Grid& g, const Fields& f, const Particles& p, long long n, double q, double h,
                             int order, DevStatus* status, cudaStream_t st) {
    const int bs = 128;
    const unsigned nb = (unsigned)((n + bs - 1) / bs);
    if (order == 1) particles_global_kernel<1, GV, DV, T><<<nb, bs, 0, st>>>(g, f, p, n, q, h, status);
    else if (order == 2) particles_global_kernel<2, GV, DV, T><<<nb, bs, 0, st>>>(g, f, p, n, q, h, status);
    else particles_global_kernel<3, GV, DV, T><<<nb, bs, 0, st>>>(g, f, p, n, q, h, status);
}

template <class T>
static void launch_global_t(const Grid& g, const Fields& f, const Particles& p, long long n, double q, double h,
                            int order, int gather_variant, int deposit_variant, DevStatus* status, cudaStream_t st) {
    if (deposit_variant) {
        if (gather_variant) launch_global_gv<1, 1, T>(g, f, p, n, q, h, order, status, st);
        else launch_global_gv<0, 1, T>(g, f, p, n, q, h, order, status, st);
    } else {
        if (gather_variant) launch_global_gv<1, 0, T>(g, f, p, n, q, h, order, status, st);
        else launch_global_gv<0, 0, T>(g, f, p, n, q, h, order, status, st);
    }
}

void launch_particles_global(const Grid& g, const Fields& f, const Particles& p, long long n, double q, double m,
                             int order, int gather_variant, int deposit_variant, int precision, DevStatus* status,
                             cudaStream_t st) {
    if (n <= 0) return;
    const double h = q * g.dt / (2.0 * m);
    if (precision) launch_global_t<float>(g, f, p, n, q, h, order, gather_variant, deposit_variant, status, st);
    else launch_global_t<double>(g, f, p, n, q, h, order, gather_variant, deposit_variant, status, st);
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

// Along an open dimension (brick face, NEXT-1) nothing is folded: the guard layers there belong to the
// neighbouring brick and are handed over by pic_export_halo; the threads then also cover those guard layers,
// so that the exported planes are already folded along the periodic dimensions.
struct FoldRange {
    int lo[3], n[3];       // thread index range per dimension: lo .. lo + n - 1
};
__host__ __device__ inline FoldRange fold_range(const Grid& g) {
    FoldRange r;
    const int nn[3] = {g.nx, g.ny, g.nz};
    for (int d = 0; d < 3; ++d) {
        const bool open = (g.open_mask >> d) & 1;
        r.lo[d] = open ? -NG : 0;
        r.n[d] = open ? nn[d] + 2 * NG : nn[d];
    }
    return r;
}

template <int NF>
__global__ void fold_guards_kernel(Grid g, FoldRange r, double* F0, double* F1, double* F2) {
    const int i = (int)(blockIdx.x * blockDim.x + threadIdx.x) + r.lo[0];
    const int j = (int)blockIdx.y + r.lo[1], k = (int)blockIdx.z + r.lo[2];
    if (i >= r.lo[0] + r.n[0]) return;
    const bool ox = g.open_mask & 1, oy = g.open_mask & 2, oz = g.open_mask & 4;
    const bool edge = (!ox && (i < NG || i >= g.nx - NG)) || (!oy && (j < NG || j >= g.ny - NG)) ||
                      (!oz && (k < NG || k >= g.nz - NG));
    if (!edge) return;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    const int k0 = oz ? k : first_image(k, g.nz), k1 = oz ? k + 1 : g.nz + NG, kd = oz ? 1 : g.nz;
    const int j0 = oy ? j : first_image(j, g.ny), j1 = oy ? j + 1 : g.ny + NG, jd = oy ? 1 : g.ny;
    const int i0 = ox ? i : first_image(i, g.nx), i1 = ox ? i + 1 : g.nx + NG, id = ox ? 1 : g.nx;
    for (int kk = k0; kk < k1; kk += kd)
        for (int jj = j0; jj < j1; jj += jd)
            for (int ii = i0; ii < i1; ii += id) {
                const long long o = g.idx(ii, jj, kk);
                s0 += F0[o];
                if (NF == 3) { s1 += F1[o]; s2 += F2[o]; }
            }
    const long long o = g.idx(i, j, k);
    F0[o] = s0;      // distinct threads own distinct cells; a cell is an image only of itself, images are only read
    if (NF == 3) { F1[o] = s1; F2[o] = s2; }
}

void launch_fold_guards3(const Grid& g, double* F0, double* F1, double* F2, cudaStream_t st) {
    const FoldRange r = fold_range(g);
    dim3 bs(128, 1, 1), nb((r.n[0] + 127) / 128, r.n[1], r.n[2]);
    fold_guards_kernel<3><<<nb, bs, 0, st>>>(g, r, F0, F1, F2);
}

void launch_fold_guards(const Grid& g, double* F, cudaStream_t st) {
    const FoldRange r = fold_range(g);
    dim3 bs(128, 1, 1), nb((r.n[0] + 127) / 128, r.n[1], r.n[2]);
    fold_guards_kernel<1><<<nb, bs, 0, st>>>(g, r, F, nullptr, nullptr);
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

__global__ void iota_kernel(unsigned long long* id, long long n, unsigned long long base) {
    long long ip = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ip < n) id[ip] = base + (unsigned long long)ip;
}

void launch_iota(unsigned long long* id, long long n, unsigned long long base, cudaStream_t st) {
    if (n <= 0) return;
    iota_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(id, n, base);
}

}  // namespace pic
