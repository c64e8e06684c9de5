// pic_internal.h -- shared declarations of libpic_b200 (CUDA side only; never
// seen by the oracle).  Layout of the device arena, the by-value grid
// descriptor handed to kernels, and the launcher prototypes of each stage.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/pic.h"

namespace pic {

constexpr int NG = PIC_NG;          // guard cells per side
constexpr int MAX_SPECIES = 8;
constexpr double C_LIGHT = 299792458.0;       // CODATA 2018 (exact)
constexpr double EPS0 = 8.8541878128e-12;     // CODATA 2018

// Grid descriptor, passed by value to every kernel.
struct Grid {
    int nx, ny, nz;          // interior cells
    int px, py, pz;          // padded extents: px = pitch (even, >= nx + 2 NG), py = ny + 2 NG, ...
    long long sy, sz;        // strides in elements: sy = px, sz = px * py
    long long npad;          // px * py * pz elements per component
    double dx, dy, dz;
    double inv_dx, inv_dy, inv_dz;   // 1.0/dx rounded once (reading R30)
    double xmin, ymin, zmin;
    double xmax, ymax, zmax;         // xmin + nx*dx
    double Lx, Ly, Lz;               // nx*dx
    double dt;
    int open_mask;                   // bit d set: dimension d is a brick face (NEXT-1), not a periodic boundary of this grid
    __host__ __device__ inline long long idx(int i, int j, int k) const {   // interior cell index -> padded offset
        return (long long)(i + NG) + sy * (long long)(j + NG) + sz * (long long)(k + NG);
    }
};

// Nine field components, padded layout.
struct Fields {
    double *Ex, *Ey, *Ez, *Bx, *By, *Bz, *Jx, *Jy, *Jz;
};

// One SoA particle buffer.
struct Particles {
    double *x, *y, *z, *ux, *uy, *uz, *w;
    unsigned long long* id;
};

// Device-side flags and counters (one small block in the arena).
struct DevStatus {
    int ephys;                 // set by particle kernels: moved >= 1 cell or non-finite
    int ebox;                  // set by the load validator: outside the box / non-finite
    unsigned long long n_fast; // counters [0..2] of pic_get_counters
    unsigned long long n_slow;
    unsigned long long n_global;
};

// ---- yee.cu ---------------------------------------------------------------
// Six CUtensorMap objects (Ex Ey Ez Bx By Bz), kept opaque here so that only yee.cu needs <cuda.h>.
struct YeeMaps {
    alignas(64) unsigned char map[6 * 128];    // Ex Ey Ez Bx By Bz
    int valid;       // 1: the maps are built and the TMA kernels configured
};
int make_yee_maps(const Grid& g, const Fields& f, YeeMaps* out);   // 0 = ok; else the plain kernels are used
// maps == nullptr or !maps->valid: plain one-thread-per-cell kernels; else the TMA-staged tile kernels
void launch_push_B(const Grid& g, const Fields& f, double dth, const YeeMaps* maps, cudaStream_t st);
void launch_push_E(const Grid& g, const Fields& f, double dt, const YeeMaps* maps, cudaStream_t st);
void launch_fill_guards(const Grid& g, double* F, cudaStream_t st);       // periodic images of one component
// binomial (1-2-1 along x, y, z) smoothing of the interior of F, npass passes; tmp = a padded scratch component
int launch_smooth_binomial(const Grid& g, double* F, double* tmp, int npass, cudaStream_t st);

// ---- particles_global.cu --------------------------------------------------
// gather + Boris + move + Esirkepov with global fp64 atomics + wrap; any particle order.
// gather_variant: 0 = order n in every direction, 1 = order n-1 along a component's staggered directions
// deposit_variant: 0 = Esirkepov (charge-conserving), 1 = direct deposition at the middle of the move
// precision: 0 = fp64 throughout, 1 = gather and Boris push in fp32 (NEXT-4), positions and deposition in fp64
void launch_particles_global(const Grid& g, const Fields& f, const Particles& p, long long n, double q,
                             double m, int order, int gather_variant, int deposit_variant, int precision,
                             DevStatus* status, cudaStream_t st);
void launch_deposit_rho(const Grid& g, const Particles& p, long long n, double q, int order, double* rho_pad,
                        cudaStream_t st);
void launch_fold_guards(const Grid& g, double* F, cudaStream_t st);       // sum periodic images into the interior
void launch_fold_guards3(const Grid& g, double* F0, double* F1, double* F2, cudaStream_t st);   // three components, one launch
void launch_validate(const Grid& g, const Particles& p, long long n, DevStatus* status, cudaStream_t st);
void launch_iota(unsigned long long* id, long long n, unsigned long long base, cudaStream_t st);

// ---- bricks.cu (NEXT-1: brick decomposition) ----------------------------------
// Halo planes of a group of three components across face (dim, side): E and B export their NG interior
// boundary layers and import into the guard layers; J exports its guard layers and import ADDS them to
// the interior boundary layers.  A plane covers the full padded extent of the other two dimensions.
long long halo_doubles(const Grid& g, int dim);                    // per component and side
void launch_halo_pack(const Grid& g, const double* F, int dim, int first_layer, double* buf, cudaStream_t st);
void launch_halo_unpack(const Grid& g, double* F, int dim, int first_layer, const double* buf, bool add, cudaStream_t st);
void launch_halo_fill(const Grid& g, double* F, int dim, int first_layer, double value, cudaStream_t st);
void launch_shift_z(const Grid& g, double* F, int ncells, cudaStream_t st);          // moving window (NEXT-2)
void launch_add_plane(const Grid& g, double* F, int k, const double* values_dev, cudaStream_t st);
constexpr int DAMP_MAX = 64;                       // thickest damping layer (cells); the table travels as a kernel argument
struct DampTable {
    int n = 0;
    double f[DAMP_MAX];
};
void launch_damp_z(const Grid& g, double* F0, double* F1, double* F2, const DampTable& t, cudaStream_t st);
// Leavers of face (dim, side), in place: find_leavers appends their indices to leaver_idx (and their 8-double records
// x y z ux uy uz w id to out, if given) and counts them in counters[0] (device, zeroed by the caller; entries beyond
// `capacity` are counted but not stored); close_holes then moves the stayers among the last L places into the holes
// below n - L (tailflag, fillers: scratch of L entries each; counters[1], counters[2] zeroed by the caller).
void launch_find_leavers(const Grid& g, const Particles& p, long long n, int dim, int side, double* out,
                         long long capacity, unsigned int* leaver_idx, unsigned long long* counters, cudaStream_t st);
int launch_close_holes(const Particles& p, long long n, long long L, const unsigned int* leaver_idx, unsigned int* tailflag,
                       unsigned int* fillers, unsigned long long* counters, cudaStream_t st);
void launch_append_arrivals(const Particles& dst, long long at, const double* in, long long count, double sx, double sy,
                            double sz, cudaStream_t st);

// ---- sort.cu ----------------------------------------------------------------
// scratch: key[n] u32, rank[n] u32, block_sums[...] u32
struct SortScratch {
    unsigned int* key;
    unsigned int* rank;
    unsigned int* block_sums;
    long long block_sums_len;
};
// perm == nullptr: src is scattered into dst; else only perm[] (sorted position -> index in src) is written
// keys_in != nullptr: per-particle cell keys of src written by the last fused particle kernel (key pass skipped)
int launch_sort(const Grid& g, const Particles& src, const Particles& dst, long long n, unsigned int* cell_offset,
                unsigned int* perm, const unsigned int* keys_in, const SortScratch& sc,
                cudaStream_t st);   // returns kernels launched
void launch_apply_perm(const Particles& src, const Particles& dst, long long n, const unsigned int* perm,
                       cudaStream_t st);                     // dst[d] = src[perm[d]]
long long sort_block_sums_len(long long ncell);

// ---- particles_tile.cu ------------------------------------------------------
// fused gather + push + deposit per cell-sorted tile (shared-memory stencil, per-cell register accumulators).
struct TileScratch {
    void* ptr;
    size_t bytes;
};
// fresh = no step since the species' last sort (every particle sits in its listed cell): smaller stencil, 2 blocks/SM.
// perm != nullptr (deferred sort): sorted particle d is read from p at perm[d] and every array (w and id too)
// is written to pout at d; perm == nullptr: pout == p, in place.
// key_out != nullptr: the kernel also writes the cell key of every particle's new position (for the next pic_sort)
int launch_particles_tile(const Grid& g, const Fields& f, const Particles& p, const Particles& pout,
                          const unsigned int* perm, unsigned int* key_out, long long n, double q, double m, int order,
                          int gather_variant, int precision, const unsigned int* cell_offset, bool fresh,
                          DevStatus* status, cudaStream_t st);  // kernels launched
int tile_setup();   // one-time cudaFuncSetAttribute calls; returns cudaError_t as int

}  // namespace pic
