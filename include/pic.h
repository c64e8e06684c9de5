/*
 * pic.h -- C ABI of libpic_b200.so: the fp64 explicit electromagnetic
 * particle-in-cell (PIC) hot path on one NVIDIA B200 (sm_100a).
 *
 * What the calls follow.  PAPER.md:45 (section II) fixes the method: a
 * "fully-kinetic, electromagnetic particle-in-cell" code with "explicit
 * algorithms, which iterate forward in time"; PAPER.md:57 (section III.A)
 * fixes the figure of merit ("parallel particle-and-cell update rate per
 * second").  The five parts of one cycle -- order-1/2/3 field gather from the
 * staggered Yee grid, relativistic Boris push, Esirkepov charge-conserving
 * current deposition, Yee FDTD update of E and B, periodic per-cell counting
 * sort -- and the names pic_init_grid / pic_load_particles / pic_step /
 * pic_sort / pic_get_fields / pic_get_particles are stated in
 * BASELINE.json:north_star; their arithmetic is written out in SURVEY.md
 * section 8(c.1) and DESIGN.md ("The path", "Readings").
 *
 * Conventions common to all calls
 *   - SI units.  u = gamma*v [m/s].  c = 299792458 m/s, eps0 = 8.8541878128e-12
 *     F/m are compiled in; charge q [C] and mass m [kg] are per species.
 *   - Field arrays crossing this ABI are GUARD-FREE, nx*ny*nz doubles per
 *     component, index = i + nx*(j + ny*k) (x fastest).  All boundaries are
 *     periodic unless options say otherwise ("open_mask": faces shared with
 *     neighbouring bricks, NEXT-1; "absorb_mask": open ends, NEXT-2; both at
 *     the end of this header).  Yee staggering is implied by the component:
 *       Ex,Jx (i+1/2,j,k)   Ey,Jy (i,j+1/2,k)   Ez,Jz (i,j,k+1/2)
 *       Bx (i,j+1/2,k+1/2)  By (i+1/2,j,k+1/2)  Bz (i+1/2,j+1/2,k)
 *       rho at nodes (i,j,k); node i sits at xmin + i*dx.
 *     (Inside the library every component carries PIC_NG periodic guard cells
 *     per side; they never cross the ABI.)
 *   - Every pointer argument is tagged host or device by an *_on_device flag
 *     of the call (0 = host memory, 1 = device memory of the same GPU).
 *   - Ownership: the caller owns the device arena and the CUDA stream given
 *     to pic_init_grid and keeps both alive until pic_destroy.  The library
 *     never allocates or frees device memory; it owns only its host context.
 *     pic_load_particles / pic_set_fields copy in, pic_get_* copy out into
 *     caller buffers.
 *   - Errors: every call returns PIC_OK (0) or a negative code; no exceptions,
 *     no abort; a NULL context gives PIC_EINVAL.  pic_last_error returns a
 *     context-owned string describing the last failure.
 *   - All device work is enqueued on the context's stream.  pic_step and
 *     pic_sort are asynchronous; pic_get_*, pic_deposit_rho, pic_sync and
 *     pic_get_counters synchronise that stream.
 *   - There is no CPU fallback anywhere behind this ABI.
 *
 * Beyond the six calls of BASELINE.json:north_star the header declares the
 * additions SURVEY.md 8(b) proposes (arena query, field input, rho diagnostic,
 * errors, counters, stage timers, options), the SURVEY.md 8(f) extensions --
 * NEXT-1 bricks (pic_step_stage, pic_halo_doubles, pic_export_halo,
 * pic_import_halo, pic_export_leavers, pic_import_arrivals), NEXT-2 open ends,
 * moving window and plane source (pic_shift_window, pic_add_plane), NEXT-3
 * gather / deposit variants and smoothing and the NEXT-4 mixed-precision mode
 * (all through pic_set_option) -- and the machine-rate probes pic_probe_*.
 */
#ifndef PIC_B200_H
#define PIC_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pic_ctx pic_ctx; /* opaque: one simulation on one GPU */

enum {
    PIC_OK = 0,
    PIC_EINVAL = -1, /* bad argument: order, sizes, NULL, dt above the Courant limit,
                        particle outside the box or non-finite at load              */
    PIC_ENOMEM = -2, /* arena too small / more particles than np_max               */
    PIC_ECUDA = -3,  /* CUDA runtime error (text in pic_last_error)                */
    PIC_ESTATE = -4, /* call order: step/sort/get before the species were loaded   */
    PIC_EPHYS = -5   /* raised on the device during a step: a particle moved >= 1
                        cell in one step or its position became non-finite; it is
                        reported by the next synchronising call                    */
};

#define PIC_NG 4 /* guard cells per side of every internal field array */

/* Number of entries written by pic_get_counters. */
#define PIC_NCOUNTERS 9

/* Number of entries written by pic_get_stage_ms. */
#define PIC_NSTAGES 8

/*
 * Bytes of device arena pic_init_grid needs.  Pure function of its arguments
 * (no CUDA call).  np_max[s] = capacity of species s (particles); the library
 * holds two SoA copies of every species (out-of-place sort).
 * Errors: PIC_EINVAL (nx,ny,nz < 1, order not in 1..3, nspecies not in 1..8,
 * np_max[s] < 0 or >= 2^31, NULL pointers).
 */
int pic_query_arena(int nx, int ny, int nz, int order, int nspecies,
                    const long long* np_max /*host*/, size_t* bytes /*host*/);

/*
 * Create a simulation (SURVEY 8(c.1) "State at the start of step n").
 *   nx,ny,nz        cells per dimension (= unknowns per field component)
 *   dx,dy,dz        cell sizes [m] (> 0);  xmin,ymin,zmin  position of node 0
 *   dt              time step [s], 0 < dt <= 1/(c*sqrt(1/dx^2+1/dy^2+1/dz^2))
 *                   (3-D Courant limit, reading R17), else PIC_EINVAL
 *   order           B-spline degree of the particle shape, 1, 2 or 3 (R4)
 *   nspecies, np_max[s]   as in pic_query_arena
 *   arena_dev, arena_bytes  DEVICE memory, 256-byte aligned, >= pic_query_arena
 *   cuda_stream     a cudaStream_t (NULL = legacy default stream)
 * All fields start at zero and every species is empty.  The arena is zeroed
 * asynchronously on the stream.
 */
int pic_init_grid(pic_ctx** out, int nx, int ny, int nz, double dx, double dy, double dz,
                  double xmin, double ymin, double zmin, double dt, int order, int nspecies,
                  const long long* np_max /*host*/, void* arena_dev, size_t arena_bytes,
                  void* cuda_stream);

/*
 * Overwrite E^n and B^n (both at integer time, reading R1).  Any pointer may
 * be NULL (= that component becomes zero).  Guard-free arrays (see top);
 * the library refreshes its periodic guard cells.
 */
int pic_set_fields(pic_ctx*, const double* Ex, const double* Ey, const double* Ez,
                   const double* Bx, const double* By, const double* Bz, int src_on_device);

/*
 * Replace the content of species `species` by n particles: positions x,y,z [m]
 * inside [min, min + N*d), momenta ux,uy,uz = gamma*v [m/s] taken as
 * u^{n-1/2} (R9: no backward half-push is applied), weights w (real particles
 * per macro-particle).  Particle p receives id = p (its load index), which
 * travels with it through every sort.  The species becomes "unsorted".
 * Errors: PIC_EINVAL (species index, n < 0, NULL with n > 0, a position
 * outside the box or non-finite -- checked on the device, the call
 * synchronises), PIC_ENOMEM (n > np_max[species]).
 */
int pic_load_particles(pic_ctx*, int species, double q, double m, long long n,
                       const double* x, const double* y, const double* z,
                       const double* ux, const double* uy, const double* uz,
                       const double* w, int src_on_device);

/*
 * Advance nsteps PIC cycles (SURVEY 8(c.1) steps 1-8 per cycle):
 *   J := 0;  for every species: gather E,B at x^n (order-n B-splines read at
 *   the Yee locations), Boris push u^{n-1/2} -> u^{n+1/2}, move
 *   x~ = x + dt*u/gamma, Esirkepov deposition of J^{n+1/2} from (x^n, x~),
 *   periodic wrap;  B -= (dt/2) curl E;  E += dt (c^2 curl B - J/eps0);
 *   B -= (dt/2) curl E.
 * Correct for ANY particle order; a species that has been sorted (pic_sort)
 * and is still close to sorted (option "drift_watch") runs the fused per-tile
 * kernel, anything else the global-atomic path; both evaluate the same
 * expressions per particle, so the path only changes summation order in J.
 * Asynchronous.  Errors: PIC_ESTATE (no species
 * loaded), PIC_EINVAL (nsteps < 0), PIC_ECUDA.
 */
int pic_step(pic_ctx*, int nsteps);

/*
 * Counting sort of every loaded species by cell key = i + nx*(j + ny*k),
 * (i,j,k) = clamp(floor((x - xmin)/dx), 0, nx-1) etc. of the stored position:
 * histogram, exclusive scan, and the move of x,y,z,ux,uy,uz,w,id into the
 * second SoA buffer with a buffer swap.  Afterwards keys are non-decreasing in
 * container order (as seen by pic_get_particles / pic_get_cell_offsets); the
 * order inside one cell is unspecified (R24).  By default (option
 * "sort_deferred") only the permutation is computed here and the move is
 * carried out by the next reader of the container -- normally the fused
 * per-tile kernel of the next pic_step, which reads its inputs through the
 * permutation at no extra pass over the data; the observable result is the
 * same.  Asynchronous.
 * What not sorting costs (one B200, round 2/3 measurements, DESIGN.md section
 * 6): the fused kernel is fastest on the step right after a sort; sorting every
 * step costs 1.4 ms at 134 M particles and the step then takes 31.0 ms, while
 * a species that drifts for four steps runs the slower "drift" instantiation:
 * configs[1] 8.2 ms per step sorted every 4 steps against 7.0 ms sorted every
 * step, configs[3] 15.0 against 7.4 ms, configs[4] 50.7 against 33.4 ms.  A
 * caller that does not need a particular cadence should sort every step, or
 * set the option "auto_sort" and let pic_step do it.
 */
int pic_sort(pic_ctx*);

/*
 * Copy out E^n, B^n and the J^{n+1/2} of the last step (zeros before the
 * first), guard-free.  NULL = skip that component.  Synchronises.
 */
int pic_get_fields(pic_ctx*, double* Ex, double* Ey, double* Ez, double* Bx, double* By,
                   double* Bz, double* Jx, double* Jy, double* Jz, int dst_on_device);

/*
 * Copy out species `species` in container order.  *n (host) receives the
 * particle count; every array pointer may be NULL (= skip) and otherwise has
 * room for that many entries (call once with all-NULL arrays to learn n).
 * id = load index.  Synchronises.
 */
int pic_get_particles(pic_ctx*, int species, long long* n /*host*/, double* x, double* y,
                      double* z, double* ux, double* uy, double* uz, double* w,
                      unsigned long long* id, int dst_on_device);

/*
 * Diagnostic (not on the step path): nodal charge density
 * rho[i,j,k] = sum_p q w/(dx dy dz) S(xi-i) S(eta-j) S(zeta-k), same order as
 * the simulation, of one species (species >= 0) or of all (-1).  nx*ny*nz
 * doubles, guard-free.  Synchronises.
 */
int pic_deposit_rho(pic_ctx*, int species, double* rho, int dst_on_device);

/*
 * Copy out the cell offsets of the last pic_sort of `species`:
 * nx*ny*nz + 1 unsigned 32-bit entries, offset[c] = first container index of
 * cell c, offset[ncell] = n.  PIC_ESTATE if the species was never sorted.
 */
int pic_get_cell_offsets(pic_ctx*, int species, unsigned int* offsets, int dst_on_device);

/*
 * Device counters since pic_init_grid (host array of PIC_NCOUNTERS unsigned
 * 64-bit values).  Synchronises.
 *   [0] particle updates done by the fused per-tile kernel (fast deposit path)
 *   [1] particle updates done by the fused kernel's in-tile slow path
 *       (particle crossed a cell face or was not in its listed cell)
 *   [2] particle updates done with global atomics (unsorted species, or a
 *       particle found outside its tile's halo)
 *   [3] kernels launched by the library
 *   [4] steps completed     [5] sorts completed
 *   [6] 1 = the TMA-staged Yee kernels run (default), 0 = the tensor maps could not be
 *       built at pic_init_grid and pic_step runs the plain Yee kernels (same
 *       values, about 40 % slower); pic_last_error right after pic_init_grid
 *       then holds a warning
 *   [7] particle launches that ran the global-atomic kernel for a SORTED
 *       species because the drift watch (option "drift_watch") found it stale
 *   [8] particles deleted at open ends ("absorb_mask") and by pic_shift_window
 */
int pic_get_counters(pic_ctx*, unsigned long long* counters /*host*/);

/*
 * Per-stage device time, in milliseconds, summed over every pic_step iteration
 * and every pic_sort issued since stage timing was switched on
 * (pic_set_option("stage_timing",1)) or since the previous pic_get_stage_ms,
 * whichever is later.  CUDA events are recorded on the context's stream around
 * each stage; pic_step / pic_sort never wait on them, so timing does not
 * serialise the host with the device.  Host array of PIC_NSTAGES floats:
 *   [0] zero J   [1] particles (gather+push+deposit, all species)
 *   [2] J guard fold   [3] Yee B (both half pushes)   [4] Yee E
 *   [5] sort (all species)   [6] step iterations summed   [7] sorts summed
 * Synchronises and resets the sums.  PIC_ESTATE if stage timing is off.
 */
int pic_get_stage_ms(pic_ctx*, float* ms /*host*/);

/*
 * Options (all default 0 unless stated):
 *   "stage_timing"   1 = record CUDA events around every stage of pic_step
 *   "force_path"     0 = automatic, 1 = always the global-atomic particle
 *                    kernel, 2 = always the fused per-tile kernel (requires a
 *                    prior pic_sort, else PIC_ESTATE at pic_step)
 *   "yee_tma"        bit 0 = B push, bit 1 = E push through the TMA-staged
 *                    tile kernels; 3 (default) = both, 0 = plain one-thread-
 *                    per-cell kernels (same arithmetic, bit-identical result)
 *   "tile_fresh"     1 (default) = a species that has not stepped since its
 *                    last pic_sort runs the small-stencil, two-blocks-per-SM
 *                    variant of the fused per-tile kernel; 0 = always the
 *                    drift-tolerant variant (same arithmetic per particle)
 *   "sort_deferred"  1 (default) = pic_sort writes only the permutation (4 B per
 *                    particle); the particle data are moved by the next fused
 *                    per-tile kernel, which reads its inputs through the
 *                    permutation and writes its outputs in sorted order (any
 *                    other reader -- pic_get_particles, the global-atomic
 *                    kernel -- triggers the move first); 0 = pic_sort moves
 *                    the data itself.  Same result either way.
 *   "fuse_keys"      1 (default) = the fused per-tile kernel also writes every
 *                    particle's new cell key, so that the next pic_sort
 *                    skips its pass over the positions; 0 = pic_sort always
 *                    computes the keys itself
 *   "auto_sort"      k > 0 = pic_step (and stage 0 of pic_step_stage) sorts by
 *                    itself, exactly as pic_sort would, before any step on which
 *                    a loaded species is unsorted or has taken k steps since its
 *                    last sort; 1 keeps every step on the fused kernel's fastest
 *                    instantiation.  The container order then changes inside
 *                    pic_step, the values do not (beyond summation order).
 *                    0 (default) = only the caller sorts.
 *   "drift_watch"    1 (default) = after every fused-kernel launch the library
 *                    reads back (asynchronously, never waiting) how many
 *                    particles left the fast per-cell deposit path; a species
 *                    that lost more than 20 % of them since its last pic_sort
 *                    runs the global-atomic kernel until it is sorted again
 *                    (the fused kernel deposits such particles one per warp
 *                    iteration, which is slower than global atomics).  The
 *                    values computed do not depend on the path beyond
 *                    summation order.  0 = a sorted species always runs the
 *                    fused kernel.  Ignored while force_path != 0.
 *   "gather_variant" 0 (default) = the gather uses the same shape order n in every
 *                    direction (reading R5); 1 = the "energy-conserving" gather:
 *                    order n-1 along every direction in which the gathered
 *                    component is staggered (
 *                    oracle: ora_gather_variant).  Both particle kernels.
 *   "precision"      0 (default) = fp64 throughout (the contract of BASELINE.json);
 *                    1 = mixed precision (NEXT-4; oracle: ora_gather_f32,
 *                    ora_boris_f32): field values and shape weights are rounded
 *                    to fp32 for the gather, the gather and the Boris push run
 *                    in fp32, momenta are stored as doubles holding fp32 values;
 *                    positions, the move, the deposition and the Yee update
 *                    stay fp64 (charge conservation is untouched).  Tolerances
 *                    against the oracle are those of fp32 arithmetic.
 *   "deposit_variant" 0 (default) = Esirkepov charge-conserving deposition; 1 =
 *                    direct deposition (NEXT-3; oracle: ora_deposit_direct): q w v
 *                    of the move, spread with the order-n shape at the middle
 *                    of the move at each component's Yee location.  NOT charge
 *                    conserving.  Runs in the global-atomic kernel only (a sorted
 *                    species leaves the fused per-tile kernel while it is set).
 *   "smooth_passes"  k >= 0 (default 0, at most 16): after deposition and guard
 *                    fold, each J component is filtered k times by the periodic
 *                    binomial (1/4, 1/2, 1/4) stencil along x, then y, then z
 *                    (NEXT-3; oracle: ora_smooth_binomial).  Not on a brick.
 *   "open_mask"      bit d set = dimension d of this grid ends at faces shared
 *                    with neighbouring bricks instead of wrapping onto itself
 *                    (NEXT-1, below): particles are not wrapped along d, J guard
 *                    layers along d are not folded, and pic_step is replaced by
 *                    pic_step_stage plus the halo calls.  Default 0.
 *   "absorb_mask"    bit d set = both faces normal to dimension d are OPEN ENDS
 *                    (NEXT-2): every field value beyond them is zero at all times,
 *                    current deposited beyond them is dropped, and a particle that
 *                    leaves through them is deleted at the end of the particle
 *                    stage (which then synchronises; any number of them: the
 *                    deletion works in batches of np_max / 3).  Implies the same
 *                    bits of "open_mask", in whichever order the two options are
 *                    set (a later "open_mask" keeps them); pic_step stays
 *                    available when every open dimension is absorbing.  Oracle:
 *                    OracleSim(open_z=True).
 *   "id_base"        ids given by the next pic_load_particles start at this
 *                    value (default 0), so that bricks can hand out disjoint ids.
 * Unknown name: PIC_EINVAL.  Like every call that takes a context it makes the
 * context's device current and returns the sticky error, if one is pending.
 */
int pic_set_option(pic_ctx*, const char* name, long long value);

/*
 * ---- NEXT-1: brick decomposition -------
 * Every brick is its own context over its own block of cells (xmin etc. of
 * pic_init_grid are the brick's).  Along a dimension named in "open_mask" the
 * NG = PIC_NG guard layers stand for the neighbour's cells.  One step of a brick
 * is, in this order (paper_2303_12873_b200/bricks.py drives it):
 *   pic_step_stage(0)   J := 0, gather + push + deposit, J fold along the periodic
 *                       dimensions
 *   J halos             pic_export_halo(2, d, side) -> neighbour's
 *                       pic_import_halo(2, d, 1 - side): SUM into its interior
 *   particles           pic_export_leavers / pic_import_arrivals per open
 *                       dimension, one dimension after the other; then pic_sort
 *   pic_step_stage(1)   first B half push;  B halos (group 1: copy into guards)
 *   pic_step_stage(2)   E push;             E halos (group 0)
 *   pic_step_stage(3)   second B half push; B halos; the step counter advances
 * E and B halos are also exchanged once after pic_set_fields.  Exchanging the
 * dimensions one after the other (planes cover the full padded extent of the
 * other two dimensions) carries the edges and corners along.
 *
 * pic_halo_doubles: doubles of one halo message (three components, NG layers)
 *   across a face normal to `dim`; -1 on a bad argument.
 * pic_export_halo / pic_import_halo: group 0 = E, 1 = B, 2 = J; side 0 = the face
 *   at the low end of `dim`, 1 = the high end; buf = DEVICE buffer of
 *   pic_halo_doubles(dim) doubles, written / read on the context's stream.
 *   E, B: export the NG interior layers next to the face, import into the guard
 *   layers beyond it.  J: export the guard layers, import ADDS to the interior
 *   layers.  PIC_EINVAL if the brick has fewer than NG cells along dim.
 * pic_export_leavers: particles of `species` with position < min (side 0) or
 *   >= max (side 1) along dim are removed from the container and written to
 *   buf (DEVICE, 8 doubles each: x y z ux uy uz w and the id's bit pattern);
 *   *count = how many.  PIC_ENOMEM (container unchanged) if more than
 *   `capacity` (or a third of the species' np_max, the size of the library's
 *   index scratch) leave.  In place: one coordinate of every particle is read,
 *   the holes are filled from the end of the container.  Synchronises once.  The
 *   species counts as unsorted afterwards.
 * pic_import_arrivals: appends `count` such records, their positions shifted by
 *   (shift_x, shift_y, shift_z) (the box length when the face is the periodic
 *   seam of the whole domain, else 0).  PIC_ENOMEM if they do not fit np_max.
 */
int pic_step_stage(pic_ctx*, int stage);

/*
 * ---- NEXT-2: moving window and antenna -----------
 * pic_shift_window: the box moves up by `ncells` cells along z (needs
 *   "absorb_mask" bit 2): field index k now names what was k + ncells, the top
 *   ncells planes are new and zero, zmin grows by ncells*dz, particles below the
 *   new zmin are deleted (*deleted = how many, may be NULL; no limit on the
 *   number -- unlike pic_export_leavers the deletion works in batches of
 *   np_max / 3), every species counts as unsorted.  Fresh plasma for the new planes is the caller's to append with
 *   pic_import_arrivals.  Synchronises.
 * pic_add_plane: F[:, :, k] += values for one component (0..8 = Ex Ey Ez Bx By Bz
 *   Jx Jy Jz), values = nx*ny doubles, x fastest (host or device).  An antenna is
 *   pic_step_stage(0), pic_add_plane(6.., k, J_source), pic_step_stage(1..3).
 * pic_set_damping: an absorbing layer of `ncells` planes in front of each open z
 *   end (needs absorb_mask bit 2, else PIC_ESTATE).  factors[m] (HOST, ncells
 *   doubles, copied) multiplies every value of B after each B half push and of E
 *   after the E push on the plane m cells from the face (m = 0 next to it), at
 *   both ends; the caller chooses the profile, e.g. exp(-a ((n - m)/n)^2).
 *   ncells = 0 removes the layers.  PIC_EINVAL: ncells not in 0 .. 64, layers
 *   that overlap (2 ncells > nz), a factor that is not finite.
 */
int pic_shift_window(pic_ctx*, int ncells, long long* deleted /*host, may be NULL*/);
int pic_add_plane(pic_ctx*, int component, int k, const double* values, int src_on_device);
int pic_set_damping(pic_ctx*, int ncells, const double* factors /*host*/);
long long pic_halo_doubles(pic_ctx*, int dim);
int pic_export_halo(pic_ctx*, int group, int dim, int side, double* buf_dev);
int pic_import_halo(pic_ctx*, int group, int dim, int side, const double* buf_dev);
int pic_export_leavers(pic_ctx*, int species, int dim, int side, double* buf_dev, long long capacity,
                       long long* count /*host*/);
int pic_import_arrivals(pic_ctx*, int species, const double* buf_dev, long long count, double shift_x,
                        double shift_y, double shift_z);

/* Wait for the context's stream; returns a pending PIC_EPHYS / PIC_ECUDA. */
int pic_sync(pic_ctx*);

/* Context-owned, valid until the next call on this context.  NULL ctx gives a
 * static string. */
const char* pic_last_error(pic_ctx*);

/* Free the host context (the arena and the stream stay the caller's). */
int pic_destroy(pic_ctx*);

/* Library version string, e.g. "pic_b200 0.1 (sm_100a)". */
const char* pic_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PIC_B200_H */
