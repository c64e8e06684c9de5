/*
 * pic_oracle.c -- ORACLE (test infrastructure, NOT the product).  See
 * pic_oracle.h for scope, conventions and citations.  Plain loops, modulo
 * indexing, no guards, no tiles, no blocking, no fusion.  Build with
 *   gcc -O2 -ffp-contract=off -shared -fPIC -o libpic_oracle.so pic_oracle.c -lm
 */
#include "pic_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define ORA_C    299792458.0        /* m/s,  CODATA 2018 (exact)  */
#define ORA_EPS0 8.8541878128e-12   /* F/m,  CODATA 2018          */

/* deposit / gather window half-width: h = 1 for n = 1, h = 2 for n = 2,3.
 * Window of node indices [i0 - h, i0 + h + 1] with i0 = floor(xi of the OLD
 * position).  It contains the support of S^n at the old position, at a new
 * position less than one cell away, and at both staggerings (offset 0 and
 * 1/2); extra nodes evaluate to exact zeros (reading R7). */
static int window_h(int n) { return 1 + n / 2; }
#define WMAX 6  /* 2*h + 2 at h = 2 */

double ora_const_c(void) { return ORA_C; }
double ora_const_eps0(void) { return ORA_EPS0; }

/* Centred cardinal B-splines (SURVEY 8(c.1) "Shape function"):
 *  S1(r) = max(0, 1-|r|)
 *  S2(r) = 3/4 - r^2 (|r|<=1/2);  (3/2-|r|)^2/2 (1/2<|r|<=3/2);  0 else
 *  S3(r) = 2/3 - r^2 + |r|^3/2 (|r|<=1);  (2-|r|)^3/6 (1<|r|<=2);  0 else  */
double ora_shape(int n, double r)
{
    double a = fabs(r);
    if (n == 1) {
        return a < 1.0 ? 1.0 - a : 0.0;
    } else if (n == 2) {
        if (a <= 0.5) return 0.75 - a * a;
        if (a <= 1.5) { double t = 1.5 - a; return 0.5 * t * t; }
        return 0.0;
    } else if (n == 3) {
        if (a <= 1.0) return 2.0 / 3.0 - a * a + 0.5 * a * a * a;
        if (a <= 2.0) { double t = 2.0 - a; return t * t * t / 6.0; }
        return 0.0;
    }
    return NAN;
}

double ora_courant_dt(const ora_grid* g)
{
    return 1.0 / (ORA_C * sqrt(1.0 / (g->dx * g->dx) + 1.0 / (g->dy * g->dy) +
                               1.0 / (g->dz * g->dz)));
}

static long long imod(long long a, long long n)
{
    long long r = a % n;
    return r < 0 ? r + n : r;
}

static size_t gidx(const ora_grid* g, long long i, long long j, long long k)
{
    return (size_t)(imod(i, g->nx) +
                    (long long)g->nx * (imod(j, g->ny) + (long long)g->ny * imod(k, g->nz)));
}

/* one component with staggering offsets (ox,oy,oz) in {0, 1/2}:
 * F_p = sum_{ijk} S(xi-i-ox) S(eta-j-oy) S(zeta-k-oz) F[i mod nx, j mod ny, k mod nz] */
static double gather_one(const ora_grid* g, int n, double xi, double eta, double zeta,
                         double ox, double oy, double oz, const double* F)
{
    int h = window_h(n), wn = 2 * h + 2;
    long long i0 = (long long)floor(xi), j0 = (long long)floor(eta), k0 = (long long)floor(zeta);
    double sum = 0.0;
    for (int c = 0; c < wn; ++c) {
        long long k = k0 - h + c;
        double sz = ora_shape(n, zeta - (double)k - oz);
        for (int b = 0; b < wn; ++b) {
            long long j = j0 - h + b;
            double sy = ora_shape(n, eta - (double)j - oy);
            for (int a = 0; a < wn; ++a) {
                long long i = i0 - h + a;
                double sx = ora_shape(n, xi - (double)i - ox);
                sum += sx * sy * sz * F[gidx(g, i, j, k)];
            }
        }
    }
    return sum;
}

int ora_gather(const ora_grid* g, int order, long long np,
               const double* x, const double* y, const double* z,
               const double* Ex, const double* Ey, const double* Ez,
               const double* Bx, const double* By, const double* Bz,
               double* Exp, double* Eyp, double* Ezp,
               double* Bxp, double* Byp, double* Bzp)
{
    if (order < 1 || order > 3) return -1;
    double inv_dx = 1.0 / g->dx, inv_dy = 1.0 / g->dy, inv_dz = 1.0 / g->dz;
    for (long long p = 0; p < np; ++p) {
        double xi = (x[p] - g->xmin) * inv_dx;
        double eta = (y[p] - g->ymin) * inv_dy;
        double zeta = (z[p] - g->zmin) * inv_dz;
        Exp[p] = gather_one(g, order, xi, eta, zeta, 0.5, 0.0, 0.0, Ex);
        Eyp[p] = gather_one(g, order, xi, eta, zeta, 0.0, 0.5, 0.0, Ey);
        Ezp[p] = gather_one(g, order, xi, eta, zeta, 0.0, 0.0, 0.5, Ez);
        Bxp[p] = gather_one(g, order, xi, eta, zeta, 0.0, 0.5, 0.5, Bx);
        Byp[p] = gather_one(g, order, xi, eta, zeta, 0.5, 0.0, 0.5, By);
        Bzp[p] = gather_one(g, order, xi, eta, zeta, 0.5, 0.5, 0.0, Bz);
    }
    return 0;
}

/* ---- NEXT-3 (8(c.2) item 5): gather variants --------------------------------
 * variant 0: the same order n in every direction (ora_gather, reading R5).
 * variant 1: "energy-conserving" / Galerkin gather: along every direction in which the
 *   component is STAGGERED the shape order is n-1, along the others n:
 *   Ex_p = sum S^{n-1}(xi-i-1/2) S^n(eta-j) S^n(zeta-k) Ex[i,j,k], Bx_p = sum S^n(xi-i)
 *   S^{n-1}(eta-j-1/2) S^{n-1}(zeta-k-1/2) Bx[i,j,k], and cyclic permutations.
 * S^0 is the top-hat on the half-open interval [-1/2, 1/2) (so that a particle on a cell
 * boundary belongs to the cell floor(xi) puts it in). */
double ora_shape0(double r) { return (r >= -0.5 && r < 0.5) ? 1.0 : 0.0; }

static double shape_any(int n, double r) { return n == 0 ? ora_shape0(r) : ora_shape(n, r); }

/* one component, staggering offsets (ox,oy,oz) in {0, 1/2}, per-direction orders (n1,n2,n3) */
static double gather_one_orders(const ora_grid* g, int n, int n1, int n2, int n3, double xi, double eta,
                                double zeta, double ox, double oy, double oz, const double* F)
{
    int h = window_h(n), wn = 2 * h + 2;      /* the order-n window contains every lower-order support */
    long long i0 = (long long)floor(xi), j0 = (long long)floor(eta), k0 = (long long)floor(zeta);
    double sum = 0.0;
    for (int c = 0; c < wn; ++c) {
        long long k = k0 - h + c;
        double sz = shape_any(n3, zeta - (double)k - oz);
        for (int b = 0; b < wn; ++b) {
            long long j = j0 - h + b;
            double sy = shape_any(n2, eta - (double)j - oy);
            for (int a = 0; a < wn; ++a) {
                long long i = i0 - h + a;
                double sx = shape_any(n1, xi - (double)i - ox);
                sum += sx * sy * sz * F[gidx(g, i, j, k)];
            }
        }
    }
    return sum;
}

int ora_gather_variant(const ora_grid* g, int order, int variant, long long np,
                       const double* x, const double* y, const double* z,
                       const double* Ex, const double* Ey, const double* Ez,
                       const double* Bx, const double* By, const double* Bz,
                       double* Exp, double* Eyp, double* Ezp,
                       double* Bxp, double* Byp, double* Bzp)
{
    if (order < 1 || order > 3 || variant < 0 || variant > 1) return -1;
    if (variant == 0)
        return ora_gather(g, order, np, x, y, z, Ex, Ey, Ez, Bx, By, Bz, Exp, Eyp, Ezp, Bxp, Byp, Bzp);
    int n = order, m = order - 1;             /* m: order along a staggered direction */
    double inv_dx = 1.0 / g->dx, inv_dy = 1.0 / g->dy, inv_dz = 1.0 / g->dz;
    for (long long p = 0; p < np; ++p) {
        double xi = (x[p] - g->xmin) * inv_dx;
        double eta = (y[p] - g->ymin) * inv_dy;
        double zeta = (z[p] - g->zmin) * inv_dz;
        Exp[p] = gather_one_orders(g, n, m, n, n, xi, eta, zeta, 0.5, 0.0, 0.0, Ex);
        Eyp[p] = gather_one_orders(g, n, n, m, n, xi, eta, zeta, 0.0, 0.5, 0.0, Ey);
        Ezp[p] = gather_one_orders(g, n, n, n, m, xi, eta, zeta, 0.0, 0.0, 0.5, Ez);
        Bxp[p] = gather_one_orders(g, n, n, m, m, xi, eta, zeta, 0.0, 0.5, 0.5, Bx);
        Byp[p] = gather_one_orders(g, n, m, n, m, xi, eta, zeta, 0.5, 0.0, 0.5, By);
        Bzp[p] = gather_one_orders(g, n, m, m, n, xi, eta, zeta, 0.5, 0.5, 0.0, Bz);
    }
    return 0;
}

/* NEXT-3: binomial (1-2-1) smoothing of one field component, periodic, `npass` passes; one pass
 * filters along x, then y, then z: F'[i] = F[i-1]/4 + F[i]/2 + F[i+1]/4. */
int ora_smooth_binomial(const ora_grid* g, int npass, double* F)
{
    if (npass < 0) return -1;
    size_t n = (size_t)g->nx * g->ny * g->nz;
    double* T = (double*)malloc(n * sizeof(double));
    if (!T) return -2;
    for (int pass = 0; pass < npass; ++pass)
        for (int d = 0; d < 3; ++d) {
            for (long long k = 0; k < g->nz; ++k)
                for (long long j = 0; j < g->ny; ++j)
                    for (long long i = 0; i < g->nx; ++i) {
                        size_t lo = gidx(g, i - (d == 0), j - (d == 1), k - (d == 2));
                        size_t hi = gidx(g, i + (d == 0), j + (d == 1), k + (d == 2));
                        T[gidx(g, i, j, k)] = 0.25 * F[lo] + 0.5 * F[gidx(g, i, j, k)] + 0.25 * F[hi];
                    }
            memcpy(F, T, n * sizeof(double));
        }
    free(T);
    return 0;
}

/* ---- NEXT-4: mixed precision -- fp32 fields and momenta, fp64 positions ----------------
 * The gather and the Boris push run in IEEE single precision; everything that touches a position (shape
 * arguments, the move, the deposition) stays in double.
 *  gather: the shape values are evaluated in double (they are functions of the fp64 position) and rounded to
 *   float; the field values are rounded to float; products and the sum are float, in the same loop order as
 *   ora_gather:  F_p = sum_k sum_j sum_i  fl(fl(fl(sx*sy)*sz) * F).
 *  Boris: the formulas of ora_boris with every variable and constant a float (h, 1/c^2 rounded once from
 *   double); momenta come in and go out as doubles that hold float values. */
static float gather_one_f32(const ora_grid* g, int n, int n1, int n2, int n3, double xi, double eta, double zeta,
                            double ox, double oy, double oz, const double* F)
{
    int h = window_h(n), wn = 2 * h + 2;
    long long i0 = (long long)floor(xi), j0 = (long long)floor(eta), k0 = (long long)floor(zeta);
    float sum = 0.0f;
    for (int c = 0; c < wn; ++c) {
        long long k = k0 - h + c;
        float sz = (float)shape_any(n3, zeta - (double)k - oz);
        for (int b = 0; b < wn; ++b) {
            long long j = j0 - h + b;
            float sy = (float)shape_any(n2, eta - (double)j - oy);
            for (int a = 0; a < wn; ++a) {
                long long i = i0 - h + a;
                float sx = (float)shape_any(n1, xi - (double)i - ox);
                float t = sx * sy;
                t = t * sz;
                t = t * (float)F[gidx(g, i, j, k)];
                sum = sum + t;
            }
        }
    }
    return sum;
}

int ora_gather_f32(const ora_grid* g, int order, int variant, long long np,
                   const double* x, const double* y, const double* z,
                   const double* Ex, const double* Ey, const double* Ez,
                   const double* Bx, const double* By, const double* Bz,
                   double* Exp, double* Eyp, double* Ezp,
                   double* Bxp, double* Byp, double* Bzp)
{
    if (order < 1 || order > 3 || variant < 0 || variant > 1) return -1;
    int n = order, m = variant ? order - 1 : order;
    double inv_dx = 1.0 / g->dx, inv_dy = 1.0 / g->dy, inv_dz = 1.0 / g->dz;
    for (long long p = 0; p < np; ++p) {
        double xi = (x[p] - g->xmin) * inv_dx;
        double eta = (y[p] - g->ymin) * inv_dy;
        double zeta = (z[p] - g->zmin) * inv_dz;
        Exp[p] = (double)gather_one_f32(g, n, m, n, n, xi, eta, zeta, 0.5, 0.0, 0.0, Ex);
        Eyp[p] = (double)gather_one_f32(g, n, n, m, n, xi, eta, zeta, 0.0, 0.5, 0.0, Ey);
        Ezp[p] = (double)gather_one_f32(g, n, n, n, m, xi, eta, zeta, 0.0, 0.0, 0.5, Ez);
        Bxp[p] = (double)gather_one_f32(g, n, n, m, m, xi, eta, zeta, 0.0, 0.5, 0.5, Bx);
        Byp[p] = (double)gather_one_f32(g, n, m, n, m, xi, eta, zeta, 0.5, 0.0, 0.5, By);
        Bzp[p] = (double)gather_one_f32(g, n, m, m, n, xi, eta, zeta, 0.5, 0.5, 0.0, Bz);
    }
    return 0;
}

int ora_boris_f32(long long np, double q, double m, double dt,
                  double* ux, double* uy, double* uz,
                  const double* Exp, const double* Eyp, const double* Ezp,
                  const double* Bxp, const double* Byp, const double* Bzp)
{
    float h = (float)(q * dt / (2.0 * m));
    float inv_c2 = (float)(1.0 / (ORA_C * ORA_C));
    for (long long p = 0; p < np; ++p) {
        float ex = (float)Exp[p], ey = (float)Eyp[p], ez = (float)Ezp[p];
        float bx = (float)Bxp[p], by = (float)Byp[p], bz = (float)Bzp[p];
        float umx = (float)ux[p] + h * ex;
        float umy = (float)uy[p] + h * ey;
        float umz = (float)uz[p] + h * ez;
        float gam = sqrtf(1.0f + (umx * umx + umy * umy + umz * umz) * inv_c2);
        float tx = h * bx / gam, ty = h * by / gam, tz = h * bz / gam;
        float t2 = tx * tx + ty * ty + tz * tz;
        float sx = 2.0f * tx / (1.0f + t2), sy = 2.0f * ty / (1.0f + t2), sz = 2.0f * tz / (1.0f + t2);
        float upx = umx + (umy * tz - umz * ty);
        float upy = umy + (umz * tx - umx * tz);
        float upz = umz + (umx * ty - umy * tx);
        float uqx = umx + (upy * sz - upz * sy);
        float uqy = umy + (upz * sx - upx * sz);
        float uqz = umz + (upx * sy - upy * sx);
        ux[p] = (double)(uqx + h * ex);
        uy[p] = (double)(uqy + h * ey);
        uz[p] = (double)(uqz + h * ez);
    }
    return 0;
}

/* Boris (1970), relativistic form:
 *  h = q dt/(2m); u- = u + h E; gamma- = sqrt(1+|u-|^2/c^2); t = h B/gamma-;
 *  s = 2t/(1+|t|^2); u' = u- + u- x t; u+ = u- + u' x s; u_new = u+ + h E. */
int ora_boris(long long np, double q, double m, double dt,
              double* ux, double* uy, double* uz,
              const double* Exp, const double* Eyp, const double* Ezp,
              const double* Bxp, const double* Byp, const double* Bzp)
{
    double h = q * dt / (2.0 * m);
    double inv_c2 = 1.0 / (ORA_C * ORA_C);
    for (long long p = 0; p < np; ++p) {
        double umx = ux[p] + h * Exp[p];
        double umy = uy[p] + h * Eyp[p];
        double umz = uz[p] + h * Ezp[p];
        double gam = sqrt(1.0 + (umx * umx + umy * umy + umz * umz) * inv_c2);
        double tx = h * Bxp[p] / gam, ty = h * Byp[p] / gam, tz = h * Bzp[p] / gam;
        double t2 = tx * tx + ty * ty + tz * tz;
        double sx = 2.0 * tx / (1.0 + t2), sy = 2.0 * ty / (1.0 + t2), sz = 2.0 * tz / (1.0 + t2);
        double upx = umx + (umy * tz - umz * ty);
        double upy = umy + (umz * tx - umx * tz);
        double upz = umz + (umx * ty - umy * tx);
        double uqx = umx + (upy * sz - upz * sy);
        double uqy = umy + (upz * sx - upx * sz);
        double uqz = umz + (upx * sy - upy * sx);
        ux[p] = uqx + h * Exp[p];
        uy[p] = uqy + h * Eyp[p];
        uz[p] = uqz + h * Ezp[p];
    }
    return 0;
}

/* gamma from u^{n+1/2}; x~ = x + dt*u/gamma, unwrapped. */
int ora_move(long long np, double dt,
             const double* x, const double* y, const double* z,
             const double* ux, const double* uy, const double* uz,
             double* x1, double* y1, double* z1)
{
    double inv_c2 = 1.0 / (ORA_C * ORA_C);
    for (long long p = 0; p < np; ++p) {
        double gam = sqrt(1.0 + (ux[p] * ux[p] + uy[p] * uy[p] + uz[p] * uz[p]) * inv_c2);
        x1[p] = x[p] + dt * ux[p] / gam;
        y1[p] = y[p] + dt * uy[p] / gam;
        z1[p] = z[p] + dt * uz[p] / gam;
    }
    return 0;
}

/* Esirkepov, Comput. Phys. Commun. 135 (2001) 144:
 *  S0_d[m] = S(xi0_d - m), S1_d[m] = S(xi1_d - m), DS_d = S1_d - S0_d (nodal),
 *  Wx[i,j,k] = DSx[i] (S0y[j]S0z[k] + DSy[j]S0z[k]/2 + S0y[j]DSz[k]/2 + DSy[j]DSz[k]/3)
 *  and cyclic; Jx[i+1/2,j,k] += -(q w/(dt dy dz)) sum_{i'<=i} Wx[i',j,k], etc. */
int ora_deposit_esirkepov(const ora_grid* g, int order, long long np,
                          double q, double dt, const double* w,
                          const double* x0, const double* y0, const double* z0,
                          const double* x1, const double* y1, const double* z1,
                          double* Jx, double* Jy, double* Jz)
{
    if (order < 1 || order > 3) return -1;
    int h = window_h(order), wn = 2 * h + 2;
    double inv_dx = 1.0 / g->dx, inv_dy = 1.0 / g->dy, inv_dz = 1.0 / g->dz;
    for (long long p = 0; p < np; ++p) {
        double xi0 = (x0[p] - g->xmin) * inv_dx, xi1 = (x1[p] - g->xmin) * inv_dx;
        double et0 = (y0[p] - g->ymin) * inv_dy, et1 = (y1[p] - g->ymin) * inv_dy;
        double ze0 = (z0[p] - g->zmin) * inv_dz, ze1 = (z1[p] - g->zmin) * inv_dz;
        if (!(fabs(xi1 - xi0) < 1.0) || !(fabs(et1 - et0) < 1.0) || !(fabs(ze1 - ze0) < 1.0))
            return -5;
        long long i0 = (long long)floor(xi0), j0 = (long long)floor(et0), k0 = (long long)floor(ze0);
        double S0x[WMAX], S0y[WMAX], S0z[WMAX], DSx[WMAX], DSy[WMAX], DSz[WMAX];
        for (int a = 0; a < wn; ++a) {
            double mx = (double)(i0 - h + a), my = (double)(j0 - h + a), mz = (double)(k0 - h + a);
            S0x[a] = ora_shape(order, xi0 - mx);
            S0y[a] = ora_shape(order, et0 - my);
            S0z[a] = ora_shape(order, ze0 - mz);
            DSx[a] = ora_shape(order, xi1 - mx) - S0x[a];
            DSy[a] = ora_shape(order, et1 - my) - S0y[a];
            DSz[a] = ora_shape(order, ze1 - mz) - S0z[a];
        }
        double cx = -(q * w[p] / (dt * g->dy * g->dz));
        double cy = -(q * w[p] / (dt * g->dx * g->dz));
        double cz = -(q * w[p] / (dt * g->dx * g->dy));
        /* Jx: prefix sum along i for every (j,k) */
        for (int c = 0; c < wn; ++c)
            for (int b = 0; b < wn; ++b) {
                double acc = 0.0;
                for (int a = 0; a < wn; ++a) {
                    double Wx = DSx[a] * (S0y[b] * S0z[c] + 0.5 * DSy[b] * S0z[c] +
                                          0.5 * S0y[b] * DSz[c] + DSy[b] * DSz[c] / 3.0);
                    acc += Wx;
                    Jx[gidx(g, i0 - h + a, j0 - h + b, k0 - h + c)] += cx * acc;
                }
            }
        /* Jy: prefix sum along j for every (i,k) */
        for (int c = 0; c < wn; ++c)
            for (int a = 0; a < wn; ++a) {
                double acc = 0.0;
                for (int b = 0; b < wn; ++b) {
                    double Wy = DSy[b] * (S0z[c] * S0x[a] + 0.5 * DSz[c] * S0x[a] +
                                          0.5 * S0z[c] * DSx[a] + DSz[c] * DSx[a] / 3.0);
                    acc += Wy;
                    Jy[gidx(g, i0 - h + a, j0 - h + b, k0 - h + c)] += cy * acc;
                }
            }
        /* Jz: prefix sum along k for every (i,j) */
        for (int b = 0; b < wn; ++b)
            for (int a = 0; a < wn; ++a) {
                double acc = 0.0;
                for (int c = 0; c < wn; ++c) {
                    double Wz = DSz[c] * (S0x[a] * S0y[b] + 0.5 * DSx[a] * S0y[b] +
                                          0.5 * S0x[a] * DSy[b] + DSx[a] * DSy[b] / 3.0);
                    acc += Wz;
                    Jz[gidx(g, i0 - h + a, j0 - h + b, k0 - h + c)] += cz * acc;
                }
            }
    }
    return 0;
}

/* NEXT-3: direct, NOT charge-conserving deposition.  The particle is taken at the middle of its
 * move, x_h = (x0 + x1)/2, with the velocity of the move v = (x1 - x0)/dt, and its current q w v / dV is spread with
 * the order-n shape evaluated at each component's own Yee location:
 *  Jx[i+1/2,j,k] += (q w vx/dV) S(xi_h - i - 1/2) S(eta_h - j)       S(zeta_h - k)
 *  Jy[i,j+1/2,k] += (q w vy/dV) S(xi_h - i)       S(eta_h - j - 1/2) S(zeta_h - k)
 *  Jz[i,j,k+1/2] += (q w vz/dV) S(xi_h - i)       S(eta_h - j)       S(zeta_h - k - 1/2)     */
int ora_deposit_direct(const ora_grid* g, int order, long long np,
                       double q, double dt, const double* w,
                       const double* x0, const double* y0, const double* z0,
                       const double* x1, const double* y1, const double* z1,
                       double* Jx, double* Jy, double* Jz)
{
    if (order < 1 || order > 3) return -1;
    int h = window_h(order), wn = 2 * h + 2;
    double inv_dx = 1.0 / g->dx, inv_dy = 1.0 / g->dy, inv_dz = 1.0 / g->dz;
    double inv_dv = 1.0 / (g->dx * g->dy * g->dz);
    for (long long p = 0; p < np; ++p) {
        double xh = 0.5 * (x0[p] + x1[p]), yh = 0.5 * (y0[p] + y1[p]), zh = 0.5 * (z0[p] + z1[p]);
        double vx = (x1[p] - x0[p]) / dt, vy = (y1[p] - y0[p]) / dt, vz = (z1[p] - z0[p]) / dt;
        double xi = (xh - g->xmin) * inv_dx, eta = (yh - g->ymin) * inv_dy, zeta = (zh - g->zmin) * inv_dz;
        long long i0 = (long long)floor(xi), j0 = (long long)floor(eta), k0 = (long long)floor(zeta);
        double qw = q * w[p] * inv_dv;
        for (int c = 0; c < wn; ++c)
            for (int b = 0; b < wn; ++b)
                for (int a = 0; a < wn; ++a) {
                    long long i = i0 - h + a, j = j0 - h + b, k = k0 - h + c;
                    double sxn = ora_shape(order, xi - (double)i), sxs = ora_shape(order, xi - (double)i - 0.5);
                    double syn = ora_shape(order, eta - (double)j), sys = ora_shape(order, eta - (double)j - 0.5);
                    double szn = ora_shape(order, zeta - (double)k), szs = ora_shape(order, zeta - (double)k - 0.5);
                    size_t o = gidx(g, i, j, k);
                    Jx[o] += qw * vx * sxs * syn * szn;
                    Jy[o] += qw * vy * sxn * sys * szn;
                    Jz[o] += qw * vz * sxn * syn * szs;
                }
    }
    return 0;
}

/* one wrap suffices since |move| < 1 cell. */
static double wrap1(double v, double lo, double hi, double L)
{
    if (v >= hi) v = v - L;
    else if (v < lo) v = v + L;
    if (v == hi) v = lo; /* v = lo - tiny rounds up to hi after + L */
    return v;
}

int ora_wrap(const ora_grid* g, long long np, double* x, double* y, double* z)
{
    double Lx = g->nx * g->dx, Ly = g->ny * g->dy, Lz = g->nz * g->dz;
    double xmax = g->xmin + Lx, ymax = g->ymin + Ly, zmax = g->zmin + Lz;
    for (long long p = 0; p < np; ++p) {
        x[p] = wrap1(x[p], g->xmin, xmax, Lx);
        y[p] = wrap1(y[p], g->ymin, ymax, Ly);
        z[p] = wrap1(z[p], g->zmin, zmax, Lz);
    }
    return 0;
}

/* Yee (1966) on the staggered grid:
 *  Bx -= dth[(Ez[i,j+1,k]-Ez)/dy - (Ey[i,j,k+1]-Ey)/dz]
 *  By -= dth[(Ex[i,j,k+1]-Ex)/dz - (Ez[i+1,j,k]-Ez)/dx]
 *  Bz -= dth[(Ey[i+1,j,k]-Ey)/dx - (Ex[i,j+1,k]-Ex)/dy]                 */
int ora_yee_push_B(const ora_grid* g, double dth,
                   const double* Ex, const double* Ey, const double* Ez,
                   double* Bx, double* By, double* Bz)
{
    for (long long k = 0; k < g->nz; ++k)
        for (long long j = 0; j < g->ny; ++j)
            for (long long i = 0; i < g->nx; ++i) {
                size_t o = gidx(g, i, j, k);
                size_t xp = gidx(g, i + 1, j, k), yp = gidx(g, i, j + 1, k), zp = gidx(g, i, j, k + 1);
                Bx[o] -= dth * ((Ez[yp] - Ez[o]) / g->dy - (Ey[zp] - Ey[o]) / g->dz);
                By[o] -= dth * ((Ex[zp] - Ex[o]) / g->dz - (Ez[xp] - Ez[o]) / g->dx);
                Bz[o] -= dth * ((Ey[xp] - Ey[o]) / g->dx - (Ex[yp] - Ex[o]) / g->dy);
            }
    return 0;
}

/* SURVEY 8(c.1) step 7:
 *  Ex += dt[c^2((Bz-Bz[i,j-1,k])/dy - (By-By[i,j,k-1])/dz) - Jx/eps0]
 *  Ey += dt[c^2((Bx-Bx[i,j,k-1])/dz - (Bz-Bz[i-1,j,k])/dx) - Jy/eps0]
 *  Ez += dt[c^2((By-By[i-1,j,k])/dx - (Bx-Bx[i,j-1,k])/dy) - Jz/eps0]  */
int ora_yee_push_E(const ora_grid* g, double dt,
                   double* Ex, double* Ey, double* Ez,
                   const double* Bx, const double* By, const double* Bz,
                   const double* Jx, const double* Jy, const double* Jz)
{
    double c2 = ORA_C * ORA_C;
    for (long long k = 0; k < g->nz; ++k)
        for (long long j = 0; j < g->ny; ++j)
            for (long long i = 0; i < g->nx; ++i) {
                size_t o = gidx(g, i, j, k);
                size_t xm = gidx(g, i - 1, j, k), ym = gidx(g, i, j - 1, k), zm = gidx(g, i, j, k - 1);
                Ex[o] += dt * (c2 * ((Bz[o] - Bz[ym]) / g->dy - (By[o] - By[zm]) / g->dz) - Jx[o] / ORA_EPS0);
                Ey[o] += dt * (c2 * ((Bx[o] - Bx[zm]) / g->dz - (Bz[o] - Bz[xm]) / g->dx) - Jy[o] / ORA_EPS0);
                Ez[o] += dt * (c2 * ((By[o] - By[xm]) / g->dx - (Bx[o] - Bx[ym]) / g->dy) - Jz[o] / ORA_EPS0);
            }
    return 0;
}

/* rho[i,j,k] += (q w/(dx dy dz)) S(xi-i) S(eta-j) S(zeta-k), nodal, order n. */
int ora_deposit_rho(const ora_grid* g, int order, long long np, double q,
                    const double* w,
                    const double* x, const double* y, const double* z,
                    double* rho)
{
    if (order < 1 || order > 3) return -1;
    int h = window_h(order), wn = 2 * h + 2;
    double inv_dx = 1.0 / g->dx, inv_dy = 1.0 / g->dy, inv_dz = 1.0 / g->dz;
    double inv_dv = 1.0 / (g->dx * g->dy * g->dz);
    for (long long p = 0; p < np; ++p) {
        double xi = (x[p] - g->xmin) * inv_dx;
        double eta = (y[p] - g->ymin) * inv_dy;
        double zeta = (z[p] - g->zmin) * inv_dz;
        long long i0 = (long long)floor(xi), j0 = (long long)floor(eta), k0 = (long long)floor(zeta);
        double qw = q * w[p] * inv_dv;
        for (int c = 0; c < wn; ++c)
            for (int b = 0; b < wn; ++b)
                for (int a = 0; a < wn; ++a) {
                    long long i = i0 - h + a, j = j0 - h + b, k = k0 - h + c;
                    rho[gidx(g, i, j, k)] += qw * ora_shape(order, xi - (double)i) *
                                             ora_shape(order, eta - (double)j) *
                                             ora_shape(order, zeta - (double)k);
                }
    }
    return 0;
}

static long long clampll(long long v, long long lo, long long hi)
{
    return v < lo ? lo : (v > hi ? hi : v);
}

int ora_cell_keys(const ora_grid* g, long long np,
                  const double* x, const double* y, const double* z,
                  long long* key)
{
    double inv_dx = 1.0 / g->dx, inv_dy = 1.0 / g->dy, inv_dz = 1.0 / g->dz;
    for (long long p = 0; p < np; ++p) {
        long long i = clampll((long long)floor((x[p] - g->xmin) * inv_dx), 0, g->nx - 1);
        long long j = clampll((long long)floor((y[p] - g->ymin) * inv_dy), 0, g->ny - 1);
        long long k = clampll((long long)floor((z[p] - g->zmin) * inv_dz), 0, g->nz - 1);
        key[p] = i + (long long)g->nx * (j + (long long)g->ny * k);
    }
    return 0;
}

/* The plain definition of a stable counting sort: histogram, exclusive
 * prefix, scatter in input order. */
int ora_counting_sort(long long ncell, long long np, const long long* key,
                      long long* perm, long long* cell_offset)
{
    long long* cursor = (long long*)calloc((size_t)ncell + 1, sizeof(long long));
    if (!cursor) return -2;
    for (long long c = 0; c <= ncell; ++c) cell_offset[c] = 0;
    for (long long p = 0; p < np; ++p) {
        if (key[p] < 0 || key[p] >= ncell) { free(cursor); return -1; }
        cell_offset[key[p] + 1] += 1;
    }
    for (long long c = 0; c < ncell; ++c) cell_offset[c + 1] += cell_offset[c];
    for (long long c = 0; c < ncell; ++c) cursor[c] = cell_offset[c];
    for (long long p = 0; p < np; ++p) perm[cursor[key[p]]++] = p;
    free(cursor);
    return 0;
}
