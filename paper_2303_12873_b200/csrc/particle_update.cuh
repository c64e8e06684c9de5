// particle_update.cuh -- device code shared by the two particle kernels (CUDA
// path only): gather of one component from the padded global arrays, the
// general Esirkepov deposition of one particle through an "adder" (global
// fp64 atomics), and the complete
// order-independent update of one particle against the GLOBAL arrays.
// Follows SURVEY 8(c.1) steps 1-5 (BASELINE.json:north_star parts 1-3).
#pragma once
#include "shapes.cuh"

namespace pic {

// ---------------------------------------------------------------- gather ----
__device__ __forceinline__ double fma_t(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float fma_t(float a, float b, float c) { return fmaf(a, b, c); }

// One component: sum over the (NX+1)(NY+1)(NZ+1) support, factored z(y(x)).  The orders may differ per
// direction (gather variant 1, below).  T = arithmetic type: double, or float in the mixed-precision mode
// (field values and weights rounded to float, float FMAs).
template <int NX, int NY, int NZ, class T>
__device__ __forceinline__ T gather_comp(const double* __restrict__ F, const Grid& g, int fx, int fy, int fz,
                                         const T (&wx)[NX + 1], const T (&wy)[NY + 1], const T (&wz)[NZ + 1]) {
    const double* base = F + g.idx(fx, fy, fz);
    T acc = T(0);
#pragma unroll
    for (int c = 0; c <= NZ; ++c) {
        T accy = T(0);
#pragma unroll
        for (int b = 0; b <= NY; ++b) {
            const double* row = base + b * g.sy + c * g.sz;
            T accx = T(0);
#pragma unroll
            for (int a = 0; a <= NX; ++a) accx = fma_t(wx[a], (T)__ldg(row + a), accx);
            accy = fma_t(wy[b], accx, accy);
        }
        acc = fma_t(wz[c], accy, acc);
    }
    return acc;
}

// Gather variants (pic_set_option "gather_variant"):
//   GV = 0  the same order N in every direction (reading R5)
//   GV = 1  "energy-conserving" (Galerkin): order N - 1 along every direction in which the component is staggered
template <int N, int GV>
struct GatherOrders {
    static constexpr int NS = GV ? N - 1 : N;      // order along a staggered direction
};

// shape weights in the arithmetic type of the gather: evaluated in double (they are functions of the fp64
// position), then rounded
template <int N, class T>
__device__ __forceinline__ int shape_weights_t(double xi, T (&w)[N + 1]) {
    double wd[N + 1];
    const int f = shape_weights<N>(xi, wd);
#pragma unroll
    for (int a = 0; a <= N; ++a) w[a] = (T)wd[a];
    return f;
}

// All six components from the padded GLOBAL arrays.
template <int N, int GV, class T>
__device__ __forceinline__ void gather6_global(const Grid& g, const Fields& f, double xi, double et, double ze,
                                               T (&eb)[6]) {
    constexpr int NS = GatherOrders<N, GV>::NS;
    T wxn[N + 1], wyn[N + 1], wzn[N + 1], wxs[NS + 1], wys[NS + 1], wzs[NS + 1];
    const int fxn = shape_weights_t<N, T>(xi, wxn), fyn = shape_weights_t<N, T>(et, wyn), fzn = shape_weights_t<N, T>(ze, wzn);
    const int fxs = shape_weights_t<NS, T>(xi - 0.5, wxs), fys = shape_weights_t<NS, T>(et - 0.5, wys),
              fzs = shape_weights_t<NS, T>(ze - 0.5, wzs);
    eb[0] = gather_comp<NS, N, N, T>(f.Ex, g, fxs, fyn, fzn, wxs, wyn, wzn);
    eb[1] = gather_comp<N, NS, N, T>(f.Ey, g, fxn, fys, fzn, wxn, wys, wzn);
    eb[2] = gather_comp<N, N, NS, T>(f.Ez, g, fxn, fyn, fzs, wxn, wyn, wzs);
    eb[3] = gather_comp<N, NS, NS, T>(f.Bx, g, fxn, fys, fzs, wxn, wys, wzs);
    eb[4] = gather_comp<NS, N, NS, T>(f.By, g, fxs, fyn, fzs, wxs, wyn, wzs);
    eb[5] = gather_comp<NS, NS, N, T>(f.Bz, g, fxs, fys, fzn, wxs, wys, wzn);
}

// Esirkepov deposition of one particle through an adder:
//   Jx[i+1/2,j,k] += cx * sum_{i'<=i} DSx[i'] (S0y[j] S0z[k] + DSy[j] S0z[k]/2 + S0y[j] DSz[k]/2 + DSy[j] DSz[k]/3)
// written as cx * PDx[i] * (S0z[k] Ay[j] + DSz[k] By[j]),  A = S0 + DS/2,  B = S0/2 + DS/3.
// add(comp, ix, iy, iz, v) receives NODE indices (ix may be -2 .. nx+2) and must be atomic.
// Zero contributions are skipped, so only the (N+1)(N+2)^2 live points cost an atomic.
template <int N, class Adder>
__device__ __forceinline__ void deposit_esirkepov(const Grid& g, double xi0, double et0, double ze0, double xi1,
                                                  double et1, double ze1, double qw, bool& bad, Adder add) {
    constexpr int W = N + 3;
    double s0x[W], dsx[W], s0y[W], dsy[W], s0z[W], dsz[W];
    const int nx0 = esirkepov_shapes<N>(xi0, xi1, s0x, dsx, bad);
    const int ny0 = esirkepov_shapes<N>(et0, et1, s0y, dsy, bad);
    const int nz0 = esirkepov_shapes<N>(ze0, ze1, s0z, dsz, bad);
    if (bad) return;
    const double inv_dt = 1.0 / g.dt;
    const double cx = -qw * inv_dt * g.inv_dy * g.inv_dz;
    const double cy = -qw * inv_dt * g.inv_dx * g.inv_dz;
    const double cz = -qw * inv_dt * g.inv_dx * g.inv_dy;
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
                        if (v != 0.0) add(0, nx0 + a, ny0 + b, nz0 + c, v);
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
                        if (v != 0.0) add(1, nx0 + a, ny0 + b, nz0 + c, v);
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
                        if (v != 0.0) add(2, nx0 + a, ny0 + b, nz0 + c, v);
                    }
                }
            }
    }
}

// Adder onto the padded global J arrays: one REDG.E.ADD.F64 per live point.
struct GlobalAdder {
    double* J[3];
    long long sy, sz;
    __device__ __forceinline__ void operator()(int comp, int ix, int iy, int iz, double v) const {
        atomicAdd(J[comp] + ((long long)(ix + NG) + sy * (long long)(iy + NG) + sz * (long long)(iz + NG)), v);
    }
};

template <int N>
__device__ __forceinline__ void deposit_global(const Grid& g, const Fields& f, double xi0, double et0, double ze0,
                                               double xi1, double et1, double ze1, double qw, bool& bad) {
    GlobalAdder add{{f.Jx, f.Jy, f.Jz}, g.sy, g.sz};
    deposit_esirkepov<N>(g, xi0, et0, ze0, xi1, et1, ze1, qw, bad, add);
}

// Direct, not charge-conserving deposition (pic_set_option "deposit_variant" = 1): the particle at
// the middle of its move with the velocity of the move, order-N shapes at each component's Yee location, one
// global fp64 atomic per non-zero point.
template <int N>
__device__ __forceinline__ void deposit_direct_global(const Grid& g, const Fields& f, double x0, double y0, double z0,
                                                      double x1, double y1, double z1, double qw) {
    const double xh = 0.5 * (x0 + x1), yh = 0.5 * (y0 + y1), zh = 0.5 * (z0 + z1);
    const double inv_dt = 1.0 / g.dt;
    const double xi = (xh - g.xmin) * g.inv_dx, et = (yh - g.ymin) * g.inv_dy, ze = (zh - g.zmin) * g.inv_dz;
    double wxn[N + 1], wyn[N + 1], wzn[N + 1], wxs[N + 1], wys[N + 1], wzs[N + 1];
    const int fxn = shape_weights<N>(xi, wxn), fyn = shape_weights<N>(et, wyn), fzn = shape_weights<N>(ze, wzn);
    const int fxs = shape_weights<N>(xi - 0.5, wxs), fys = shape_weights<N>(et - 0.5, wys),
              fzs = shape_weights<N>(ze - 0.5, wzs);
    const double c = qw * (g.inv_dx * g.inv_dy * g.inv_dz);
    const double cx = c * ((x1 - x0) * inv_dt), cy = c * ((y1 - y0) * inv_dt), cz = c * ((z1 - z0) * inv_dt);
    double* jx = f.Jx + g.idx(fxs, fyn, fzn);
    double* jy = f.Jy + g.idx(fxn, fys, fzn);
    double* jz = f.Jz + g.idx(fxn, fyn, fzs);
#pragma unroll
    for (int cc = 0; cc <= N; ++cc)
#pragma unroll
        for (int b = 0; b <= N; ++b)
#pragma unroll
            for (int a = 0; a <= N; ++a) {
                const long long o = a + b * g.sy + cc * g.sz;
                const double vx = cx * wxs[a] * wyn[b] * wzn[cc], vy = cy * wxn[a] * wys[b] * wzn[cc],
                             vz = cz * wxn[a] * wyn[b] * wzs[cc];
                if (vx != 0.0) atomicAdd(jx + o, vx);
                if (vy != 0.0) atomicAdd(jy + o, vy);
                if (vz != 0.0) atomicAdd(jz + o, vz);
            }
}

// Device function used by both particle paths: the whole update of one
// particle against the GLOBAL field arrays.  DV = 0: Esirkepov deposition; 1: direct deposition.
template <int N, int GV, int DV = 0, class T = double>
__device__ __forceinline__ void update_particle_global(const Grid& g, const Fields& f, const Particles& p,
                                                       long long ip, double q, double h, DevStatus* status) {
    const double x = p.x[ip], y = p.y[ip], z = p.z[ip];
    double ux = p.ux[ip], uy = p.uy[ip], uz = p.uz[ip];
    const double w = p.w[ip];
    // normalised coordinates: a subtraction then a multiplication (R30)
    const double xi = (x - g.xmin) * g.inv_dx, et = (y - g.ymin) * g.inv_dy, ze = (z - g.zmin) * g.inv_dz;
    // step 1: gather, step 2: Boris -- in T (float in the mixed-precision mode: momenta are then doubles that hold floats)
    T eb[6];
    gather6_global<N, GV, T>(g, f, xi, et, ze, eb);
    const double inv_c2 = 1.0 / (C_LIGHT * C_LIGHT);
    {
        T tx = (T)ux, ty = (T)uy, tz = (T)uz;
        boris_push<T>((T)h, (T)inv_c2, tx, ty, tz, eb[0], eb[1], eb[2], eb[3], eb[4], eb[5]);
        ux = (double)tx; uy = (double)ty; uz = (double)tz;
    }
    // step 3: move (unwrapped)
    const double dtg = dt_over_gamma(g.dt, inv_c2, ux, uy, uz);
    const double x1 = x + dtg * ux, y1 = y + dtg * uy, z1 = z + dtg * uz;
    // step 4: deposit from (x^n, x~^{n+1})
    const double xi1 = (x1 - g.xmin) * g.inv_dx, et1 = (y1 - g.ymin) * g.inv_dy, ze1 = (z1 - g.zmin) * g.inv_dz;
    bool bad = !(isfinite(x1) && isfinite(y1) && isfinite(z1));
    if constexpr (DV == 1) {
        bad = bad || !(fabs(xi1 - xi) < 1.0) || !(fabs(et1 - et) < 1.0) || !(fabs(ze1 - ze) < 1.0);
        if (!bad && q != 0.0) deposit_direct_global<N>(g, f, x, y, z, x1, y1, z1, q * w);
    } else {
        if (!bad && q != 0.0) deposit_global<N>(g, f, xi, et, ze, xi1, et1, ze1, q * w, bad);
    }
    if (bad) atomicOr(&status->ephys, 1);
    // step 5: wrap and store
    p.x[ip] = wrap1(x1, g.xmin, g.xmax, g.Lx, g.open_mask & 1);
    p.y[ip] = wrap1(y1, g.ymin, g.ymax, g.Ly, g.open_mask & 2);
    p.z[ip] = wrap1(z1, g.zmin, g.zmax, g.Lz, g.open_mask & 4);
    p.ux[ip] = ux;
    p.uy[ip] = uy;
    p.uz[ip] = uz;
}

}  // namespace pic
