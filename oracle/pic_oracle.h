/*
 * pic_oracle.h -- ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, single-threaded fp64 CPU implementation of one explicit
 * electromagnetic particle-in-cell (PIC) cycle.  It exists only so that the
 * CUDA path can be checked against it.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares
 * no code with paper_2303_12873_b200/csrc.
 *
 * What it follows.  PAPER.md:45 (section II) fixes only the method family
 * ("fully-kinetic, electromagnetic particle-in-cell ... explicit algorithms,
 * which iterate forward in time"); PAPER.md:57 (section III.A) fixes the
 * figure of merit (particle-and-cell updates per second).  The five named
 * parts (order-1/2/3 gather from the staggered Yee grid, relativistic Boris
 * push, Esirkepov deposition, Yee FDTD, per-cell counting sort) come from
 * BASELINE.json:north_star and are written here from their textbook
 * definitions in the notation of SURVEY.md section 8(c.1); every reading of a
 * silent point is listed in DESIGN.md ("Readings").
 *
 * Conventions (DESIGN.md "Readings" R1-R12):
 *   - SI units; u = gamma*v [m/s]; c and eps0 are CODATA 2018.
 *   - Field arrays are guard-free, nx*ny*nz, index = i + nx*(j + ny*k), all
 *     boundaries periodic (indices taken modulo N).
 *   - Yee staggering: Ex,Jx (i+1/2,j,k)  Ey,Jy (i,j+1/2,k)  Ez,Jz (i,j,k+1/2)
 *                     Bx (i,j+1/2,k+1/2) By (i+1/2,j,k+1/2) Bz (i+1/2,j+1/2,k)
 *                     rho at nodes (i,j,k); node i sits at xmin + i*dx.
 *   - Normalised coordinate xi = (x - xmin) * inv_dx with inv_dx = 1.0/dx
 *     rounded once (a subtraction then a multiplication; build with
 *     -ffp-contract=off so no FMA is formed).
 *   - Shape order n = degree of the centred cardinal B-spline, n in {1,2,3}.
 *
 * Every function is pinned by tests/test_oracle_*.py against closed forms and
 * invariants (no function is "parity unpinned").
 */
#ifndef PIC_ORACLE_H
#define PIC_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int nx, ny, nz;          /* cells per dimension (= unknowns per component) */
    double dx, dy, dz;       /* cell sizes [m]                                 */
    double xmin, ymin, zmin; /* position of node 0 [m]                         */
} ora_grid;

/* speed of light and vacuum permittivity used by the oracle (CODATA 2018) */
double ora_const_c(void);
double ora_const_eps0(void);

/* S^n(r): centred cardinal B-spline of degree n (n = 1,2,3), r in cell units. */
double ora_shape(int n, double r);

/* 3-D Courant limit dt_max = 1/(c*sqrt(1/dx^2+1/dy^2+1/dz^2)). */
double ora_courant_dt(const ora_grid* g);

/* Step 1: gather E,B at the particles (6 outputs of length np).  Returns 0. */
int ora_gather(const ora_grid* g, int order, long long np,
               const double* x, const double* y, const double* z,
               const double* Ex, const double* Ey, const double* Ez,
               const double* Bx, const double* By, const double* Bz,
               double* Exp, double* Eyp, double* Ezp,
               double* Bxp, double* Byp, double* Bzp);

/* NEXT-3.  S^0: top-hat on [-1/2, 1/2). */
double ora_shape0(double r);

/* Gather variants.  variant 0 = ora_gather (same order n everywhere).  variant 1 =
 * "energy-conserving" (Galerkin) gather: order n-1 along every direction in which the component
 * is staggered, order n along the others.  Returns 0, -1 on a bad order / variant. */
int ora_gather_variant(const ora_grid* g, int order, int variant, long long np,
                       const double* x, const double* y, const double* z,
                       const double* Ex, const double* Ey, const double* Ez,
                       const double* Bx, const double* By, const double* Bz,
                       double* Exp, double* Eyp, double* Ezp,
                       double* Bxp, double* Byp, double* Bzp);

/* Binomial (1-2-1) smoothing of one component in place, periodic; one pass = x, then y, then z. */
int ora_smooth_binomial(const ora_grid* g, int npass, double* F);

/* NEXT-4: mixed precision.  ora_gather_f32 = the gather (either variant) with shape values and
 * field values rounded to float and float products / sums; ora_boris_f32 = ora_boris in float arithmetic.
 * Momenta and gathered fields travel as doubles holding float values.  Positions are never touched by them. */
int ora_gather_f32(const ora_grid* g, int order, int variant, long long np,
                   const double* x, const double* y, const double* z,
                   const double* Ex, const double* Ey, const double* Ez,
                   const double* Bx, const double* By, const double* Bz,
                   double* Exp, double* Eyp, double* Ezp,
                   double* Bxp, double* Byp, double* Bzp);
int ora_boris_f32(long long np, double q, double m, double dt,
                  double* ux, double* uy, double* uz,
                  const double* Exp, const double* Eyp, const double* Ezp,
                  const double* Bxp, const double* Byp, const double* Bzp);

/* Step 2: relativistic Boris push, u^{n-1/2} -> u^{n+1/2}, in place. */
int ora_boris(long long np, double q, double m, double dt,
              double* ux, double* uy, double* uz,
              const double* Exp, const double* Eyp, const double* Ezp,
              const double* Bxp, const double* Byp, const double* Bzp);

/* Step 3: x~^{n+1} = x^n + dt*u/gamma(u), NOT wrapped. */
int ora_move(long long np, double dt,
             const double* x, const double* y, const double* z,
             const double* ux, const double* uy, const double* uz,
             double* x1, double* y1, double* z1);

/* Step 4: Esirkepov deposition of one species, ACCUMULATED into Jx,Jy,Jz.
 * (x0,y0,z0) = x^n (inside the box), (x1,y1,z1) = unwrapped x~^{n+1};
 * |move| < 1 cell per dimension is required: returns -5 if violated. */
int ora_deposit_esirkepov(const ora_grid* g, int order, long long np,
                          double q, double dt, const double* w,
                          const double* x0, const double* y0, const double* z0,
                          const double* x1, const double* y1, const double* z1,
                          double* Jx, double* Jy, double* Jz);

/* NEXT-3: direct (not charge-conserving) deposition, ACCUMULATED into Jx,Jy,Jz: q w v S(x_half - node)/dV with
 * x_half = (x0 + x1)/2, v = (x1 - x0)/dt, order-n shapes at each component's Yee location. */
int ora_deposit_direct(const ora_grid* g, int order, long long np,
                       double q, double dt, const double* w,
                       const double* x0, const double* y0, const double* z0,
                       const double* x1, const double* y1, const double* z1,
                       double* Jx, double* Jy, double* Jz);

/* Step 5: periodic wrap of positions into [xmin, xmax), in place. */
int ora_wrap(const ora_grid* g, long long np, double* x, double* y, double* z);

/* Steps 6/8: B -= dth * curl E (forward differences); dth = dt/2. */
int ora_yee_push_B(const ora_grid* g, double dth,
                   const double* Ex, const double* Ey, const double* Ez,
                   double* Bx, double* By, double* Bz);

/* Step 7: E += dt * (c^2 curl B (backward differences) - J/eps0). */
int ora_yee_push_E(const ora_grid* g, double dt,
                   double* Ex, double* Ey, double* Ez,
                   const double* Bx, const double* By, const double* Bz,
                   const double* Jx, const double* Jy, const double* Jz);

/* Diagnostic: nodal charge density of one species, ACCUMULATED into rho. */
int ora_deposit_rho(const ora_grid* g, int order, long long np, double q,
                    const double* w,
                    const double* x, const double* y, const double* z,
                    double* rho);

/* Per-cell key of each particle: key = i + nx*(j + ny*k),
 * (i,j,k) = clamp(floor(xi,eta,zeta)) of the stored position. */
int ora_cell_keys(const ora_grid* g, long long np,
                  const double* x, const double* y, const double* z,
                  long long* key);

/* Stable counting sort by key: perm[r] = index of the particle that lands at
 * rank r; cell_offset has ncell+1 entries (exclusive prefix of the histogram). */
int ora_counting_sort(long long ncell, long long np, const long long* key,
                      long long* perm, long long* cell_offset);

#ifdef __cplusplus
}
#endif
#endif
