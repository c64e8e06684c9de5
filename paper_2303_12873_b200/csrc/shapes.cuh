// shapes.cuh -- device-side B-spline shape factors, Boris push and Esirkepov
// building blocks shared by the particle kernels (CUDA path only).
//
// Shape factors are evaluated in their per-interval polynomial form in
// delta = xi - base (SURVEY 8(c.1) "Shape function", GPU form), which is
// algebraically identical to the centred cardinal B-spline S^n(r):
//   n=1  base=floor(xi)      {1-d, d}                                   at base, base+1
//   n=2  base=floor(xi+1/2)  {(1/2-d)^2/2, 3/4-d^2, (1/2+d)^2/2}        at base-1..base+1
//   n=3  base=floor(xi)      {(1-d)^3/6, 2/3-d^2+d^3/2,
//                             1/6+(d+d^2-d^3)/2, d^3/6}                 at base-1..base+2
#pragma once
#include "pic_internal.h"

namespace pic {

// Fills w[0..N] and returns the node index of w[0].  N = 0 (used only by the energy-conserving gather
// variant, along staggered directions at order 1): the top-hat on [-1/2, 1/2), i.e. all the weight on node
// floor(xi + 1/2).
template <int N>
__device__ __forceinline__ int shape_weights(double xi, double (&w)[N + 1]) {
    if constexpr (N == 0) {
        w[0] = 1.0;
        return __double2int_rd(xi + 0.5);
    } else if constexpr (N == 1) {
        int i = __double2int_rd(xi);
        double d = xi - (double)i;
        w[0] = 1.0 - d;
        w[1] = d;
        return i;
    } else if constexpr (N == 2) {
        int b = __double2int_rd(xi + 0.5);
        double d = xi - (double)b;
        double m = 0.5 - d, p = 0.5 + d;
        w[0] = 0.5 * m * m;
        w[1] = 0.75 - d * d;
        w[2] = 0.5 * p * p;
        return b - 1;
    } else {
        int i = __double2int_rd(xi);
        double d = xi - (double)i;
        double d2 = d * d, e = 1.0 - d;
        w[0] = e * e * e * (1.0 / 6.0);
        w[1] = (2.0 / 3.0) - d2 + 0.5 * d2 * d;
        w[2] = (1.0 / 6.0) + 0.5 * (d + d2 - d2 * d);
        w[3] = d2 * d * (1.0 / 6.0);
        return i - 1;
    }
}

// Relativistic Boris push: h = q dt/(2m).  h / gamma is taken as
// h * rsqrt(gamma^2) and 2 / (1 + t^2) as 2 * rcp(1 + t^2): a reciprocal square root is half the
// instructions of a square root plus a division, and the fused kernel is bound by instruction latency.
// Both particle kernels use this one formulation, so a particle's trajectory does not depend on
// which path updated it (a few ulp away from the oracle's sqrt/divide form; the 1-step bound is 1e-12).
__device__ __forceinline__ double rsqrt_t(double x) { return rsqrt(x); }
__device__ __forceinline__ float rsqrt_t(float x) { return rsqrtf(x); }
__device__ __forceinline__ double rcp_t(double x) { return __drcp_rn(x); }
__device__ __forceinline__ float rcp_t(float x) { return __frcp_rn(x); }

// T = double, or float for the mixed-precision mode (pic_set_option "precision" = 1): the
// same formulas in single precision.
template <class T>
__device__ __forceinline__ void boris_push(T h, T inv_c2, T& ux, T& uy, T& uz, T ex, T ey, T ez, T bx, T by, T bz) {
    const T umx = ux + h * ex, umy = uy + h * ey, umz = uz + h * ez;
    const T hg = h * rsqrt_t(T(1) + (umx * umx + umy * umy + umz * umz) * inv_c2);
    const T tx = hg * bx, ty = hg * by, tz = hg * bz;
    const T t2 = tx * tx + ty * ty + tz * tz;
    const T f = T(2) * rcp_t(T(1) + t2);      // = RN(2 / (1 + t2)): the scaling by 2 is exact
    const T sx = f * tx, sy = f * ty, sz = f * tz;
    const T upx = umx + (umy * tz - umz * ty);
    const T upy = umy + (umz * tx - umx * tz);
    const T upz = umz + (umx * ty - umy * tx);
    ux = umx + (upy * sz - upz * sy) + h * ex;
    uy = umy + (upz * sx - upx * sz) + h * ey;
    uz = umz + (upx * sy - upy * sx) + h * ez;
}

// dt / gamma(u) of the position update, as dt * rsqrt(gamma^2).
__device__ __forceinline__ double dt_over_gamma(double dt, double inv_c2, double ux, double uy, double uz) {
    return dt * rsqrt(1.0 + (ux * ux + uy * uy + uz * uz) * inv_c2);
}

// One periodic wrap.  open = this dimension is a brick face: the particle keeps its
// unwrapped position and is handed to the neighbouring brick by pic_export_leavers (NEXT-1).
__device__ __forceinline__ double wrap1(double v, double lo, double hi, double L, bool open = false) {
    if (open) return v;
    if (v >= hi) v = v - L;
    else if (v < lo) v = v + L;
    if (v == hi) v = lo;
    return v;
}

// Width of the common Esirkepov window (old and new support, |move| < 1 cell).
template <int N>
struct DepWin {
    static constexpr int W = N + 3;
};

// Old and new nodal shapes on the common window of N+3 slots; slot a <-> node
// first0 - 1 + a, where first0 = node of the first old weight.  Returns first0-1.
// s0[a] = S(xi0 - node(a)), ds[a] = S(xi1 - node(a)) - s0[a].  `bad` is set
// when the move is >= 1 cell (the window cannot hold the new support).
template <int N>
__device__ __forceinline__ int esirkepov_shapes(double xi0, double xi1, double (&s0)[N + 3], double (&ds)[N + 3],
                                                bool& bad) {
    double w0[N + 1], w1[N + 1];
    int f0 = shape_weights<N>(xi0, w0);
    int f1 = shape_weights<N>(xi1, w1);
    int s = f1 - f0;                        // -1, 0 or +1
    if (s < -1 || s > 1 || !(fabs(xi1 - xi0) < 1.0)) {
        bad = true;
        s = 0;
    }
#pragma unroll
    for (int a = 0; a < N + 3; ++a) {
        double o = (a >= 1 && a <= N + 1) ? w0[(a >= 1 && a <= N + 1) ? a - 1 : 0] : 0.0;
        // new weight k sits in slot k + 1 + s
        double nm = (a <= N) ? w1[(a <= N) ? a : 0] : 0.0;                          // s = -1: slot a <- w1[a]
        double nz = (a >= 1 && a <= N + 1) ? w1[(a >= 1 && a <= N + 1) ? a - 1 : 0] : 0.0;   // s = 0
        double np = (a >= 2) ? w1[(a >= 2) ? a - 2 : 0] : 0.0;                      // s = +1: slot a <- w1[a-2]
        double n1 = (s < 0) ? nm : ((s > 0) ? np : nz);
        s0[a] = o;
        ds[a] = n1 - o;
    }
    return f0 - 1;
}

}  // namespace pic
