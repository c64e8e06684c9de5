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
#include "shapes.cuh"

namespace pic {

// ---------------------------------------------------------------- gather ----
// One component: sum over the (N+1)^3 support, factored z(y(x)).
template <int N>
__device__ __forceinline__ double gather_comp(const double* __restrict__ F, const Grid& g, int fx, int fy, int fz,
                                              const double (&wx)[N + 1], const double (&wy)[N + 1],
                                              const double (&wz)[N + 1]) {
    const double* base = F + g.idx(fx, fy, fz);
    double acc = 0.0;
#pragma unroll
    for (int c = 0; c <= N; ++c) {
        double accy = 0.0;
#pragma unroll
        for (int b = 0; b <= N; ++b) {
            const double* row = base + b * g.sy + c * g.sz;
            double accx = 0.0;
#pragma unroll
            for (int a = 0; a <= N; ++a) accx = fma(wx[a], __ldg(row + a), accx);
            accy = fma(wy[b], accx, accy);
        }
        acc = fma(wz[c], accy, acc);
    }
    return acc;
}

// Esirkepov deposition of one particle with global atomics.
//   Jx[i+1/2,j,k] += cx * sum_{i'<=i} DSx[i'] (S0y[j] S0z[k] + DSy[j] S0z[k]/2 + S0y[j] DSz[k]/2 + DSy[j] DSz[k]/3)
// written as cx * PDx[i] * (S0z[k] Ay[j] + DSz[k] By[j]),  A = S0 + DS/2,  B = S0/2 + DS/3.
template <int N>
__device__ __forceinline__ void deposit_global(const Grid& g, const Fields& f, double xi0, double et0, double ze0,
                                               double xi1, double et1, double ze1, double qw, bool& bad) {
    constexpr int W = N + 3;
    double s0x[W], dsx[W], s0y[W], dsy[W], s0z[W], dsz[W];
    int nx0 = esirkepov_shapes<N>(xi0, xi1, s0x, dsx, bad);
    int ny0 = esirkepov_shapes<N>(et0, et1, s0y, dsy, bad);
    int nz0 = esirkepov_shapes<N>(ze0, ze1, s0z, dsz, bad);
    if (bad) return;
    const double inv_dt = 1.0 / g.dt;
    const double cx = -qw * inv_dt * g.inv_dy * g.inv_dz;
    const double cy = -qw * inv_dt * g.inv_dx * g.inv_dz;
    const double cz = -qw * inv_dt * g.inv_dx * g.inv_dy;
    const long long o = g.idx(nx0, ny0, nz0);
    // Jx
    {
        double pd[W];
        double acc = 0.0;
#pragma unroll
        for (int a = 0; a < W; ++a) { acc += dsx[a]; pd[a] = cx * acc; }
#pragma unroll
        for (int c = 0; c < W; ++c)
#pragma unroll
            for (int b = 0; b < W; ++b) {
                double t = s0z[c] * (s0y[b] + 0.5 * dsy[b]) + dsz[c] * (0.5 * s0y[b] + (1.0 / 3.0) * dsy[b]);
                if (t != 0.0) {
#pragma unroll
                    for (int a = 0; a < W - 1; ++a) {
                        double v = pd[a] * t;
                        if (v != 0.0) atomicAdd(f.Jx + o + a + b * g.sy + c * g.sz, v);
                    }
                }
            }
    }
    // Jy
    {
        double pd[W];
        double acc = 0.0;
#pragma unroll
        for (int b = 0; b < W; ++b) { acc += dsy[b]; pd[b] = cy * acc; }
#pragma unroll
        for (int c = 0; c < W; ++c)
#pragma unroll
            for (int a = 0; a < W; ++a) {
                double t = s0x[a] * (s0z[c] + 0.5 * dsz[c]) + dsx[a] * (0.5 * s0z[c] + (1.0 / 3.0) * dsz[c]);
                if (t != 0.0) {
#pragma unroll
                    for (int b = 0; b < W - 1; ++b) {
                        double v = pd[b] * t;
                        if (v != 0.0) atomicAdd(f.Jy + o + a + b * g.sy + c * g.sz, v);
                    }
                }
            }
    }
    // Jz
    {
        double pd[W];
        double acc = 0.0;
#pragma unroll
        for (int c = 0; c < W; ++c) { acc += dsz[c]; pd[c] = cz * acc; }
#pragma unroll
        for (int b = 0; b < W; ++b)
#pragma unroll
            for (int a = 0; a < W; ++a) {
                double t = s0y[b] * (s0x[a] + 0.5 * dsx[a]) + dsy[b] * (0.5 * s0x[a] + (1.0 / 3.0) * dsx[a]);
                if (t != 0.0) {
#pragma unroll
                    for (int c = 0; c < W - 1; ++c) {
                        double v = pd[c] * t;
                        if (v != 0.0) atomicAdd(f.Jz + o + a + b * g.sy + c * g.sz, v);
                    }
                }
            }
    }
}

// Device function used by both particle paths: the whole update of one
// particle against the GLOBAL field arrays.
template <int N>
__device__ __forceinline__ void update_particle_global(const Grid& g, const Fields& f, const Particles& p,
                                                       long long ip, double q, double h, DevStatus* status) {
    const double x = p.x[ip], y = p.y[ip], z = p.z[ip];
    double ux = p.ux[ip], uy = p.uy[ip], uz = p.uz[ip];
    const double w = p.w[ip];
    // normalised coordinates: a subtraction then a multiplication (R30)
    const double xi = (x - g.xmin) * g.inv_dx, et = (y - g.ymin) * g.inv_dy, ze = (z - g.zmin) * g.inv_dz;
    // step 1: gather
    double wxn[N + 1], wyn[N + 1], wzn[N + 1], wxs[N + 1], wys[N + 1], wzs[N + 1];
    const int fxn = shape_weights<N>(xi, wxn), fyn = shape_weights<N>(et, wyn), fzn = shape_weights<N>(ze, wzn);
    const int fxs = shape_weights<N>(xi - 0.5, wxs), fys = shape_weights<N>(et - 0.5, wys),
              fzs = shape_weights<N>(ze - 0.5, wzs);
    const double ex = gather_comp<N>(f.Ex, g, fxs, fyn, fzn, wxs, wyn, wzn);
    const double ey = gather_comp<N>(f.Ey, g, fxn, fys, fzn, wxn, wys, wzn);
    const double ez = gather_comp<N>(f.Ez, g, fxn, fyn, fzs, wxn, wyn, wzs);
    const double bx = gather_comp<N>(f.Bx, g, fxn, fys, fzs, wxn, wys, wzs);
    const double by = gather_comp<N>(f.By, g, fxs, fyn, fzs, wxs, wyn, wzs);
    const double bz = gather_comp<N>(f.Bz, g, fxs, fys, fzn, wxs, wys, wzn);
    // step 2: Boris
    const double inv_c2 = 1.0 / (C_LIGHT * C_LIGHT);
    boris_push(h, inv_c2, ux, uy, uz, ex, ey, ez, bx, by, bz);
    // step 3: move (unwrapped)
    const double gam = sqrt(1.0 + (ux * ux + uy * uy + uz * uz) * inv_c2);
    const double x1 = x + g.dt * ux / gam, y1 = y + g.dt * uy / gam, z1 = z + g.dt * uz / gam;
    // step 4: deposit from (x^n, x~^{n+1})
    const double xi1 = (x1 - g.xmin) * g.inv_dx, et1 = (y1 - g.ymin) * g.inv_dy, ze1 = (z1 - g.zmin) * g.inv_dz;
    bool bad = !(isfinite(x1) && isfinite(y1) && isfinite(z1));
    if (!bad && q != 0.0) deposit_global<N>(g, f, xi, et, ze, xi1, et1, ze1, q * w, bad);
    if (bad) status->ephys = 1;
    // step 5: wrap and store
    p.x[ip] = wrap1(x1, g.xmin, g.xmax, g.Lx);
    p.y[ip] = wrap1(y1, g.ymin, g.ymax, g.Ly);
    p.z[ip] = wrap1(z1, g.zmin, g.zmax, g.Lz);
    p.ux[ip] = ux;
    p.uy[ip] = uy;
    p.uz[ip] = uz;
}

template <int N>
__global__ void __launch_bounds__(128) particles_global_kernel(Grid g, Fields f, Particles p, long long n, double q,
                                                               double h, DevStatus* status) {
    long long ip = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ip < n) update_particle_global<N>(g, f, p, ip, q, h, status);
    if (ip == 0) atomicAdd(&status->n_global, (unsigned long long)n);
}

void launch_particles_global(const Grid& g, const Fields& f, const Particles& p, long long n, double q, double m,
                             int order, DevStatus* status, cudaStream_t st) {
    if (n <= 0) return;
    const double h = q * g.dt / (2.0 * m);
    const int bs = 128;
    const unsigned nb = (unsigned)((n + bs - 1) / bs);
    if (order == 1) particles_global_kernel<1><<<nb, bs, 0, st>>>(g, f, p, n, q, h, status);
    else if (order == 2) particles_global_kernel<2><<<nb, bs, 0, st>>>(g, f, p, n, q, h, status);
    else particles_global_kernel<3><<<nb, bs, 0, st>>>(g, f, p, n, q, h, status);
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
