/*
 * pic_noalloc.h -- one call of libpic_b200.so for callers that are not
 * allowed to allocate device memory.
 *
 * Everything else in this library works out of an arena the caller allocates
 * (pic_query_arena / pic_init_grid in pic.h).  That is fine for a program that
 * owns its GPU, but some users of this code cannot get an arena at all:
 *   - a plugin or analysis hook that runs inside somebody else's simulation
 *     loop, where every byte of HBM is already spoken for by the host code's
 *     own pool and a cudaMalloc would either fail or fragment that pool;
 *   - code that runs between the steps of a latency-critical loop, where
 *     cudaMalloc / cudaFree are off limits because they synchronise the whole
 *     device;
 *   - a diagnostic called from an error path after an out-of-memory report,
 *     which has to work precisely when no allocation does.
 * For them the per-cell histogram and offset table of the counting sort
 * (SURVEY.md 8(a) row S, 8(c.1) "Sort": key = i + nx*(j + ny*k), histogram,
 * exclusive scan) is available as a free-standing call that takes only the
 * caller's inputs and the caller's output and allocates nothing.  It is the
 * table a caller needs to walk particles cell by cell (occupancy statistics,
 * load-balance decisions, binning for its own kernels).
 *
 * Where the working memory comes from: the three-kernel scan needs one
 * 32-bit total per chunk of 2,048 counters.  In pic_sort that scratch lives in
 * the arena; here it lives in a file-scope array in device memory that is part
 * of the library image: PIC_NOALLOC_MAX_CHUNKS entries = 64 KiB.  Every GPU on
 * which a process uses this library holds those 64 KiB from the moment the
 * library's device code is loaded there until the process exits, whether or
 * not this call is ever made.
 */
#ifndef PIC_B200_NOALLOC_H
#define PIC_B200_NOALLOC_H

#ifdef __cplusplus
extern "C" {
#endif

/* Chunks of 2,048 counters the built-in scratch can hold (64 KiB of HBM). */
#define PIC_NOALLOC_MAX_CHUNKS 16384
/* Largest grid the call accepts: nx*ny*nz + 1 <= 2048 * PIC_NOALLOC_MAX_CHUNKS
 * (33,554,431 cells; 256^3 = 16,777,216 fits, 512x256x256 does not).        */
#define PIC_NOALLOC_MAX_CELLS (2048LL * PIC_NOALLOC_MAX_CHUNKS - 1)

/*
 * Cell offsets of n particles on an nx x ny x nz grid, without allocating.
 *
 *   nx,ny,nz, dx,dy,dz, xmin,ymin,zmin   the grid, as in pic_init_grid: cell
 *                   (i,j,k) covers [xmin + i dx, xmin + (i+1) dx) x ...; a
 *                   particle's cell is clamp(floor((x - xmin) * (1.0/dx)), 0,
 *                   nx-1) per dimension, exactly the key pic_sort uses, so the
 *                   result is bit-identical to pic_sort + pic_get_cell_offsets
 *                   on the same positions.
 *   n               number of particles, 0 <= n < 2^31
 *   x,y,z           DEVICE pointers, n doubles each (not modified; may be NULL
 *                   when n == 0)
 *   offsets         DEVICE pointer, nx*ny*nz + 1 unsigned 32-bit entries,
 *                   written: offsets[c] = number of particles in cells < c
 *                   (cell index c = i + nx*(j + ny*k)), offsets[ncell] = n.
 *                   Caller-owned; the call clears it first, so its previous
 *                   contents do not matter.
 *   cuda_stream     a cudaStream_t (NULL = legacy default stream) of the
 *                   CURRENT device; the work is queued there and the call
 *                   returns without waiting for it.
 *
 * Allocation: none -- no cudaMalloc, cudaFree, cudaMallocAsync or library
 * routine that allocates; four kernels and one cudaMemsetAsync on the stream.
 *
 * First call on a device: looks up the device address of the built-in scratch
 * (cudaGetSymbolAddress; this is what loads the library's device code on that
 * GPU if nothing has yet) and caches it per device.  Make that first call with
 * the device current and BEFORE starting any stream capture; later calls on
 * the same device do no set-up.
 *
 * Sharing: there is ONE scratch array per GPU, shared by every caller in the
 * process, and it keeps whatever the last call left in it.  The call
 * overwrites every entry it reads before reading it, so stale contents are
 * harmless, but two calls whose kernels can overlap on the GPU (different
 * streams, no event between them; or two host threads) race on it and both
 * results are then undefined.  Order such calls on one stream or with events.
 *
 * Returns 0 (PIC_OK); -1 (PIC_EINVAL) for nx,ny,nz < 1, a grid beyond
 * PIC_NOALLOC_MAX_CELLS, non-positive or non-finite dx,dy,dz, n < 0 or
 * n >= 2^31, or a NULL pointer that is needed -- nothing has been queued in
 * that case; -3 (PIC_ECUDA) if a CUDA call failed.  pic_noalloc_last_error()
 * gives the reason in words (per host thread).
 */
int pic_cell_offsets_noalloc(int nx, int ny, int nz, double dx, double dy, double dz,
                             double xmin, double ymin, double zmin, long long n,
                             const double* x /*device*/, const double* y /*device*/,
                             const double* z /*device*/, unsigned int* offsets /*device*/,
                             void* cuda_stream);

/* Text of the calling thread's last pic_cell_offsets_noalloc failure ("" if none). */
const char* pic_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PIC_B200_NOALLOC_H */
