// pic_api.cu -- the C ABI of libpic_b200.so (include/pic.h): host context,
// arena carving, call-order state machine, copies across the boundary, and
// the per-step launch sequence of SURVEY 8(c.1) steps 1-8.
#include <math.h>
#include <cmath>
#include <stdarg.h>

#include <algorithm>
#include <stdio.h>
#include <string.h>

#include <new>
#include <vector>

#include <nvtx3/nvToolsExt.h>     // header-only; ranges are no-ops unless a profiler injects itself

#include "pic_internal.h"

using namespace pic;

namespace {

struct Species {
    bool loaded = false;
    bool sorted = false;        // cell_offset valid for the current buffer (up to drift since the last sort)
    int steps_since_sort = 0;
    long long n = 0, np_max = 0;
    double q = 0.0, m = 1.0;
    int cur = 0;                // which of the two SoA buffers is live
    Particles buf[2];
    unsigned int* cell_offset = nullptr;
    // Deferred sort: pic_sort wrote only perm[] (sorted position -> index in buf[cur]); the data is permuted by
    // the next fused particle kernel (which writes buf[cur ^ 1]) or by materialize() for any other reader.
    unsigned int* perm = nullptr;
    bool perm_pending = false;
    // Written by the fused per-tile kernel: the cell key of every particle's NEW position, in the container order
    // of the buffer it wrote; the next pic_sort then skips its pass over the positions.
    unsigned int* key = nullptr;
    bool keys_valid = false;
    // Drift watch: share of the last fused-kernel launch that left the fast path (slow + global), read back
    // asynchronously; above DRIFT_LIMIT the species runs the global-atomic kernel until its next pic_sort.
    bool degraded = false;
};

// A species whose last fused-kernel launch sent more than this share of its particles down the warp-serialised
// slow path (or the global gather) is faster on the global-atomic kernel: the slow path deposits ONE particle
// per warp iteration.
constexpr double DRIFT_LIMIT = 0.20;

constexpr int NSTAGE = PIC_NSTAGES;
constexpr int EV_PER_STEP = 7, EV_PER_SORT = 2;

// one timed pic_step iteration (7 consecutive events) or one timed pic_sort (2 events)
struct TimedSpan {
    size_t first;
    int kind;   // 0 = step, 1 = sort
};

}  // namespace

struct pic_ctx {
    Grid g;
    Fields f;
    double* tmp = nullptr;      // one padded scratch component (rho, pack/unpack staging)
    DevStatus* status = nullptr;
    int order = 1, nspecies = 0;
    Species sp[MAX_SPECIES];
    SortScratch sort_scratch{};
    cudaStream_t stream = nullptr;
    char err[512] = {0};
    int sticky = PIC_OK;
    unsigned long long launches = 0, steps = 0, sorts = 0;
    // options
    int stage_timing = 0, force_path = 0, yee_tma = 3, tile_fresh = 1, sort_deferred = 1, fuse_keys = 1;
    int gather_variant = 0, smooth_passes = 0, deposit_variant = 0;      // NEXT-3 options
    int precision = 0;                              // NEXT-4: 1 = gather and Boris push in fp32
    unsigned long long id_base = 0;                 // ids given at load start here (bricks: unique across contexts)
    DampTable damp;                                 // NEXT-2: damping layers in front of the open z ends (pic_set_damping)
    int absorb_mask = 0;                            // NEXT-2: dimensions whose faces are open ends (zero exterior, particles deleted)
    unsigned long long deleted = 0;                 // particles deleted at absorbing faces / by the moving window
    YeeMaps yee_maps{};
    int device = 0;                     // ordinal of the device the arena lives on; made current by every call
    int yee_tma_ok = 0;                 // tensor maps built: the TMA-staged Yee kernels are available
    // drift watch (pinned host memory, one event): counters before the first and after each species' launch of
    // the last pic_step iteration; evaluated by a later pic_step once the event has completed, never waited on
    DevStatus* watch = nullptr;         // [MAX_SPECIES + 1]
    cudaEvent_t watch_ev = nullptr;
    int auto_sort = 0;                     // option "auto_sort": pic_step sorts a species every this many steps (0 = never)
    bool watch_armed = false;
    unsigned long long watch_sorts = 0;    // c->sorts when the snapshot was armed: a pic_sort since then voids it
    bool watch_tile[MAX_SPECIES] = {false};
    int drift_watch = 1;
    unsigned long long fallbacks = 0;   // particle launches that took the global kernel because of the watch
    std::vector<cudaEvent_t> ev_pool;   // grows on demand; never waited on inside pic_step / pic_sort
    size_t ev_used = 0;
    std::vector<TimedSpan> spans;
};

namespace {

int fail(pic_ctx* c, int code, const char* fmt, ...) {
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

int cuda_fail(pic_ctx* c, cudaError_t e, const char* what) {
    c->sticky = PIC_ECUDA;
    return fail(c, PIC_ECUDA, "CUDA error in %s: %s", what, cudaGetErrorString(e));
}

#define CU(c, call)                                         \
    do {                                                    \
        cudaError_t e_ = (call);                            \
        if (e_ != cudaSuccess) return cuda_fail(c, e_, #call); \
    } while (0)

size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

int padded_pitch(int nx) { return (nx + 2 * NG + 1) & ~1; }   // even: rows stay 16-byte aligned (TMA)

struct Layout {
    size_t status, fields, tmp, species[MAX_SPECIES], cell_offset[MAX_SPECIES], perm[MAX_SPECIES], skey[MAX_SPECIES], key, rank, block_sums,
        total;
    size_t comp_bytes, np_bytes[MAX_SPECIES];
};

int make_layout(int nx, int ny, int nz, int nspecies, const long long* np_max, Layout* L) {
    const size_t npad = (size_t)padded_pitch(nx) * (size_t)(ny + 2 * NG) * (size_t)(nz + 2 * NG);
    const size_t ncell = (size_t)nx * ny * nz;
    size_t off = 0;
    L->status = off; off += align_up(sizeof(DevStatus));
    L->comp_bytes = align_up(npad * sizeof(double));
    L->fields = off; off += 9 * L->comp_bytes;
    L->tmp = off; off += L->comp_bytes;
    long long npm = 0;
    for (int s = 0; s < nspecies; ++s) {
        L->np_bytes[s] = align_up((size_t)np_max[s] * sizeof(double));
        L->species[s] = off; off += 2 * 8 * L->np_bytes[s];
        L->cell_offset[s] = off; off += align_up((ncell + 1) * sizeof(unsigned int));
        L->perm[s] = off; off += align_up((size_t)np_max[s] * sizeof(unsigned int));
        L->skey[s] = off; off += align_up((size_t)np_max[s] * sizeof(unsigned int));
        if (np_max[s] > npm) npm = np_max[s];
    }
    L->key = off; off += align_up((size_t)npm * sizeof(unsigned int));
    L->rank = off; off += align_up((size_t)npm * sizeof(unsigned int));
    L->block_sums = off; off += align_up((size_t)sort_block_sums_len((long long)ncell) * sizeof(unsigned int));
    L->total = off;
    return 0;
}

int check_dims(int nx, int ny, int nz, int order, int nspecies, const long long* np_max) {
    if (nx < 1 || ny < 1 || nz < 1 || order < 1 || order > 3 || nspecies < 1 || nspecies > MAX_SPECIES || !np_max)
        return PIC_EINVAL;
    if ((long long)nx * ny * nz >= (1LL << 31) - 1) return PIC_EINVAL;
    // several kernels launch with gridDim.y / gridDim.z = the padded extents in y and z
    if (ny + 2 * NG > 65535 || nz + 2 * NG > 65535) return PIC_EINVAL;
    for (int s = 0; s < nspecies; ++s)
        if (np_max[s] < 0 || np_max[s] >= (1LL << 31)) return PIC_EINVAL;
    return PIC_OK;
}

// ---- pack / unpack between the padded layout and guard-free arrays --------
__global__ void pack_kernel(Grid g, const double* __restrict__ pad, double* __restrict__ flat) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.nx) return;
    const int j = blockIdx.y, k = blockIdx.z;
    flat[(long long)i + (long long)g.nx * (j + (long long)g.ny * k)] = pad[g.idx(i, j, k)];
}

__global__ void unpack_kernel(Grid g, const double* __restrict__ flat, double* __restrict__ pad) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.nx) return;
    const int j = blockIdx.y, k = blockIdx.z;
    pad[g.idx(i, j, k)] = flat[(long long)i + (long long)g.nx * (j + (long long)g.ny * k)];
}

dim3 cell_grid(const Grid& g) { return dim3((g.nx + 127) / 128, g.ny, g.nz); }

// padded component -> caller's guard-free array (host or device)
int copy_out(pic_ctx* c, const double* pad, double* dst, int on_device) {
    if (!dst) return PIC_OK;
    const size_t bytes = (size_t)c->g.nx * c->g.ny * c->g.nz * sizeof(double);
    if (on_device) {
        pack_kernel<<<cell_grid(c->g), 128, 0, c->stream>>>(c->g, pad, dst);
        ++c->launches;
    } else {
        // one strided DMA copy straight out of the padded array (rows of nx doubles, pitch px): no staging buffer, no
        // pack kernel and no synchronisation between components -- pic_get_fields waits once, at its end
        const Grid& g = c->g;
        cudaMemcpy3DParms p3 = {};
        p3.srcPtr = make_cudaPitchedPtr(const_cast<double*>(pad) + g.idx(0, 0, 0), (size_t)g.px * sizeof(double),
                                        (size_t)g.nx * sizeof(double), (size_t)g.py);
        p3.dstPtr = make_cudaPitchedPtr(dst, (size_t)g.nx * sizeof(double), (size_t)g.nx * sizeof(double), (size_t)g.ny);
        p3.extent = make_cudaExtent((size_t)g.nx * sizeof(double), (size_t)g.ny, (size_t)g.nz);
        p3.kind = cudaMemcpyDeviceToHost;
        CU(c, cudaMemcpy3DAsync(&p3, c->stream));
        (void)bytes;
    }
    return PIC_OK;
}

int copy_in(pic_ctx* c, const double* src, double* pad, int on_device) {
    const size_t bytes = (size_t)c->g.nx * c->g.ny * c->g.nz * sizeof(double);
    if (!src) {
        CU(c, cudaMemsetAsync(pad, 0, (size_t)c->g.npad * sizeof(double), c->stream));
        return PIC_OK;
    }
    if (on_device) {
        unpack_kernel<<<cell_grid(c->g), 128, 0, c->stream>>>(c->g, src, pad);
    } else {
        CU(c, cudaMemcpyAsync(c->tmp, src, bytes, cudaMemcpyHostToDevice, c->stream));
        unpack_kernel<<<cell_grid(c->g), 128, 0, c->stream>>>(c->g, c->tmp, pad);
    }
    launch_fill_guards(c->g, pad, c->stream);
    c->launches += 2;
    CU(c, cudaGetLastError());
    if (!on_device) CU(c, cudaStreamSynchronize(c->stream));
    return PIC_OK;
}

// read and clear the device flags; returns a pending PIC_EPHYS
int poll_status(pic_ctx* c) {
    DevStatus h;
    CU(c, cudaMemcpyAsync(&h, c->status, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    if (h.ephys & 2) {      // the hand-over between a producer and its consumer warp timed out (particles_tile.cu)
        c->sticky = PIC_ECUDA;
        return fail(c, PIC_ECUDA, "internal: the fused particle kernel's producer / consumer hand-over timed out; the state is not valid");
    }
    if (h.ephys) {
        int zero = 0;
        CU(c, cudaMemcpyAsync(&c->status->ephys, &zero, sizeof(int), cudaMemcpyHostToDevice, c->stream));
        CU(c, cudaStreamSynchronize(c->stream));
        return fail(c, PIC_EPHYS, "a particle moved >= 1 cell in one step or its position became non-finite");
    }
    return PIC_OK;
}

int sync_and_check(pic_ctx* c) {
    if (c->sticky != PIC_OK) return c->sticky;
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaStreamSynchronize");
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e, "kernel launch");
    return poll_status(c);
}

// n consecutive events from the pool (created on first use); returns the index of the first
bool take_events(pic_ctx* c, int n, size_t* first) {
    while (c->ev_pool.size() < c->ev_used + (size_t)n) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) return false;
        c->ev_pool.push_back(e);
    }
    *first = c->ev_used;
    c->ev_used += (size_t)n;
    return true;
}

bool use_tile_path(const pic_ctx* c, const Species& s) {
    if (c->force_path == 1 || c->deposit_variant != 0) return false;     // direct deposition lives in the global kernel only
    if (c->force_path == 2) return s.sorted;
    return s.sorted && !s.degraded;
}

// Drift watch, host side: if the counters of the last watched pic_step iteration have arrived, mark every
// species whose fused-kernel launch left the fast path for more than DRIFT_LIMIT of its particles.
void poll_watch(pic_ctx* c) {
    if (!c->watch_armed || cudaEventQuery(c->watch_ev) != cudaSuccess) {
        cudaGetLastError();      // cudaErrorNotReady is not an error
        return;
    }
    c->watch_armed = false;
    if (c->watch_sorts != c->sorts) return;    // taken before the last pic_sort: says nothing about the new order
    for (int s = 0; s < c->nspecies; ++s) {
        Species& S = c->sp[s];
        if (!c->watch_tile[s] || S.n == 0 || S.steps_since_sort == 0) continue;   // sorted since: nothing to conclude
        const DevStatus &a = c->watch[s], &b = c->watch[s + 1];
        const double off_fast = (double)((b.n_slow - a.n_slow) + (b.n_global - a.n_global));
        if (off_fast > DRIFT_LIMIT * (double)S.n) S.degraded = true;
    }
}

#define ENTER(c)                                                                   \
    do {                                                                           \
        if (!(c)) return PIC_EINVAL;                                               \
        if ((c)->sticky != PIC_OK) return (c)->sticky;                             \
        cudaError_t e_ = cudaSetDevice((c)->device);                               \
        if (e_ != cudaSuccess) return cuda_fail((c), e_, "cudaSetDevice");         \
    } while (0)

// Carry out a deferred sort for a reader other than the fused per-tile kernel.
void materialize(pic_ctx* c, Species& S) {
    if (!S.perm_pending) return;
    launch_apply_perm(S.buf[S.cur], S.buf[S.cur ^ 1], S.n, S.perm, c->stream);
    if (S.n > 0) c->launches += 1;
    S.cur ^= 1;
    S.perm_pending = false;
}

}  // namespace

extern "C" {

static void zero_absorbing_guards(pic_ctx* c, int group);

const char* pic_version(void) { return "pic_b200 0.1 (sm_100a)"; }

int pic_query_arena(int nx, int ny, int nz, int order, int nspecies, const long long* np_max, size_t* bytes) {
    if (!bytes) return PIC_EINVAL;
    int rc = check_dims(nx, ny, nz, order, nspecies, np_max);
    if (rc != PIC_OK) return rc;
    Layout L;
    make_layout(nx, ny, nz, nspecies, np_max, &L);
    *bytes = L.total;
    return PIC_OK;
}

int pic_init_grid(pic_ctx** out, int nx, int ny, int nz, double dx, double dy, double dz, double xmin, double ymin,
                  double zmin, double dt, int order, int nspecies, const long long* np_max, void* arena_dev,
                  size_t arena_bytes, void* cuda_stream) {
    if (!out) return PIC_EINVAL;
    *out = nullptr;
    int rc = check_dims(nx, ny, nz, order, nspecies, np_max);
    if (rc != PIC_OK) return rc;
    if (!(dx > 0.0) || !(dy > 0.0) || !(dz > 0.0) || !isfinite(dx) || !isfinite(dy) || !isfinite(dz) ||
        !isfinite(xmin) || !isfinite(ymin) || !isfinite(zmin))
        return PIC_EINVAL;
    const double dt_max = 1.0 / (C_LIGHT * sqrt(1.0 / (dx * dx) + 1.0 / (dy * dy) + 1.0 / (dz * dz)));
    if (!(dt > 0.0) || !(dt <= dt_max)) return PIC_EINVAL;
    if (!arena_dev || ((uintptr_t)arena_dev & 255u)) return PIC_EINVAL;
    Layout L;
    make_layout(nx, ny, nz, nspecies, np_max, &L);
    if (arena_bytes < L.total) return PIC_ENOMEM;

    pic_ctx* c = new (std::nothrow) pic_ctx();
    if (!c) return PIC_ENOMEM;
    Grid& g = c->g;
    g.nx = nx; g.ny = ny; g.nz = nz;
    g.px = padded_pitch(nx); g.py = ny + 2 * NG; g.pz = nz + 2 * NG;
    g.sy = g.px; g.sz = (long long)g.px * g.py;
    g.npad = g.sz * g.pz;
    g.dx = dx; g.dy = dy; g.dz = dz;
    g.inv_dx = 1.0 / dx; g.inv_dy = 1.0 / dy; g.inv_dz = 1.0 / dz;
    g.xmin = xmin; g.ymin = ymin; g.zmin = zmin;
    g.Lx = nx * dx; g.Ly = ny * dy; g.Lz = nz * dz;
    g.xmax = xmin + g.Lx; g.ymax = ymin + g.Ly; g.zmax = zmin + g.Lz;
    g.dt = dt;
    g.open_mask = 0;
    c->order = order;
    c->nspecies = nspecies;
    c->stream = (cudaStream_t)cuda_stream;
    {   // the device the arena lives on becomes the context's device (every later call makes it current)
        cudaPointerAttributes pa;
        if (cudaPointerGetAttributes(&pa, arena_dev) != cudaSuccess || pa.type != cudaMemoryTypeDevice ||
            cudaSetDevice(pa.device) != cudaSuccess) {
            cudaGetLastError();
            delete c;
            return PIC_EINVAL;
        }
        c->device = pa.device;
    }

    char* base = (char*)arena_dev;
    c->status = (DevStatus*)(base + L.status);
    double** comps[9] = {&c->f.Ex, &c->f.Ey, &c->f.Ez, &c->f.Bx, &c->f.By, &c->f.Bz, &c->f.Jx, &c->f.Jy, &c->f.Jz};
    for (int k = 0; k < 9; ++k) *comps[k] = (double*)(base + L.fields + (size_t)k * L.comp_bytes);
    c->tmp = (double*)(base + L.tmp);
    for (int s = 0; s < nspecies; ++s) {
        Species& S = c->sp[s];
        S.np_max = np_max[s];
        for (int b = 0; b < 2; ++b) {
            char* pb = base + L.species[s] + (size_t)b * 8 * L.np_bytes[s];
            double** arr[7] = {&S.buf[b].x, &S.buf[b].y, &S.buf[b].z, &S.buf[b].ux, &S.buf[b].uy, &S.buf[b].uz,
                               &S.buf[b].w};
            for (int a = 0; a < 7; ++a) *arr[a] = (double*)(pb + (size_t)a * L.np_bytes[s]);
            S.buf[b].id = (unsigned long long*)(pb + (size_t)7 * L.np_bytes[s]);
        }
        S.cell_offset = (unsigned int*)(base + L.cell_offset[s]);
        S.perm = (unsigned int*)(base + L.perm[s]);
        S.key = (unsigned int*)(base + L.skey[s]);
    }
    c->sort_scratch.key = (unsigned int*)(base + L.key);
    c->sort_scratch.rank = (unsigned int*)(base + L.rank);
    c->sort_scratch.block_sums = (unsigned int*)(base + L.block_sums);
    c->sort_scratch.block_sums_len = sort_block_sums_len((long long)nx * ny * nz);

    // zero the status block, the fields and the scratch component (particles are written at load)
    cudaError_t e = cudaMemsetAsync(base, 0, L.tmp + L.comp_bytes, c->stream);
    if (e == cudaSuccess) e = (cudaError_t)tile_setup();
    if (e == cudaSuccess) e = cudaMallocHost((void**)&c->watch, sizeof(DevStatus) * (MAX_SPECIES + 1));
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->watch_ev, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        if (c->watch) cudaFreeHost(c->watch);
        delete c;
        return PIC_ECUDA;
    }
    // Tensor maps for the TMA-staged Yee kernels.  A failure is not fatal (the plain kernels compute the same
    // values) but it is not silent either: pic_last_error says so and pic_get_counters[6] stays 0.
    const int yrc = make_yee_maps(c->g, c->f, &c->yee_maps);
    c->yee_tma_ok = (yrc == 0 && c->yee_maps.valid) ? 1 : 0;
    if (!c->yee_tma_ok)
        snprintf(c->err, sizeof(c->err),
                 "warning: tensor maps for the TMA-staged Yee kernels could not be built (make_yee_maps = %d); "
                 "pic_step uses the plain Yee kernels", yrc);
    *out = c;
    return PIC_OK;
}

int pic_set_fields(pic_ctx* c, const double* Ex, const double* Ey, const double* Ez, const double* Bx,
                   const double* By, const double* Bz, int src_on_device) {
    ENTER(c);
    const double* src[6] = {Ex, Ey, Ez, Bx, By, Bz};
    double* dst[6] = {c->f.Ex, c->f.Ey, c->f.Ez, c->f.Bx, c->f.By, c->f.Bz};
    for (int k = 0; k < 6; ++k) {
        int rc = copy_in(c, src[k], dst[k], src_on_device);
        if (rc != PIC_OK) return rc;
    }
    if (c->absorb_mask) {
        zero_absorbing_guards(c, 0);
        zero_absorbing_guards(c, 1);
    }
    return PIC_OK;
}

int pic_load_particles(pic_ctx* c, int species, double q, double m, long long n, const double* x, const double* y,
                       const double* z, const double* ux, const double* uy, const double* uz, const double* w,
                       int src_on_device) {
    ENTER(c);
    if (species < 0 || species >= c->nspecies) return fail(c, PIC_EINVAL, "species index %d out of range", species);
    if (n < 0 || !(m > 0.0) || !isfinite(q) || !isfinite(m)) return fail(c, PIC_EINVAL, "bad n, q or m");
    if (n > 0 && (!x || !y || !z || !ux || !uy || !uz || !w)) return fail(c, PIC_EINVAL, "NULL particle array");
    Species& S = c->sp[species];
    if (n > S.np_max) return fail(c, PIC_ENOMEM, "n = %lld exceeds np_max = %lld", n, S.np_max);
    S.cur = 0;
    S.perm_pending = false;
    S.keys_valid = false;
    Particles& P = S.buf[0];
    const double* src[7] = {x, y, z, ux, uy, uz, w};
    double* dst[7] = {P.x, P.y, P.z, P.ux, P.uy, P.uz, P.w};
    const cudaMemcpyKind kind = src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    for (int a = 0; a < 7 && n > 0; ++a)
        CU(c, cudaMemcpyAsync(dst[a], src[a], (size_t)n * sizeof(double), kind, c->stream));
    launch_iota(P.id, n, c->id_base, c->stream);
    launch_validate(c->g, P, n, c->status, c->stream);
    c->launches += (n > 0) ? 2 : 0;
    CU(c, cudaGetLastError());
    DevStatus h;
    CU(c, cudaMemcpyAsync(&h, c->status, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    S.q = q; S.m = m; S.n = n;
    S.sorted = false; S.steps_since_sort = 0; S.degraded = false;
    if (h.ebox) {
        int zero = 0;
        CU(c, cudaMemcpyAsync(&c->status->ebox, &zero, sizeof(int), cudaMemcpyHostToDevice, c->stream));
        CU(c, cudaStreamSynchronize(c->stream));
        S.loaded = false; S.n = 0;
        return fail(c, PIC_EINVAL, "species %d: a particle is outside the box or non-finite", species);
    }
    S.loaded = true;
    return PIC_OK;
}

// ---- NEXT-2: absorbing faces (zero exterior), used by the step, pic_set_fields and pic_shift_window -----
// guard layers of a group of three components := 0 along every absorbing dimension
static void zero_absorbing_guards(pic_ctx* c, int group) {
    double* F[3][3] = {{c->f.Ex, c->f.Ey, c->f.Ez}, {c->f.Bx, c->f.By, c->f.Bz}, {c->f.Jx, c->f.Jy, c->f.Jz}};
    const int n[3] = {c->g.nx, c->g.ny, c->g.nz};
    for (int d = 0; d < 3; ++d)
        if ((c->absorb_mask >> d) & 1)
            for (int k = 0; k < 3; ++k) {
                launch_halo_fill(c->g, F[group][k], d, -NG, 0.0, c->stream);
                launch_halo_fill(c->g, F[group][k], d, n[d], 0.0, c->stream);
                c->launches += 2;
            }
}

// damping layers of E (group 0) or B (group 1) after their push
static void damp_layers(pic_ctx* c, int group) {
    if (c->damp.n == 0) return;
    if (group == 0) launch_damp_z(c->g, c->f.Ex, c->f.Ey, c->f.Ez, c->damp, c->stream);
    else launch_damp_z(c->g, c->f.Bx, c->f.By, c->f.Bz, c->damp, c->stream);
    c->launches += 1;
}

// Particles of one species beyond face (dim, side) are taken out of the container in place (bricks.cu); their records go
// to out (device, 8 doubles each) if given.  More than `capacity` leavers: PIC_ENOMEM, container unchanged -- unless
// `remaining` is given: then the first `capacity` of them (in list order) are taken out and *remaining = how many are
// still in the container (discard_leavers comes back for them).  Synchronises once (the count).
static int take_leavers(pic_ctx* c, Species& S, int dim, int side, double* out, long long capacity, long long* count,
                        long long* remaining = nullptr) {
    *count = 0;
    if (remaining) *remaining = 0;
    if (!S.loaded || S.n == 0) return PIC_OK;
    materialize(c, S);
    // scratch: the sort's rank array holds the leaver list, the tail flags and the filler list (a third each)
    const long long cap = std::min<long long>(capacity, S.np_max / 3);
    unsigned int* leaver_idx = c->sort_scratch.rank;
    unsigned int* tailflag = leaver_idx + S.np_max / 3;
    unsigned int* fillers = tailflag + S.np_max / 3;
    unsigned long long* counters = reinterpret_cast<unsigned long long*>(reinterpret_cast<char*>(c->status) + 128);
    CU(c, cudaMemsetAsync(counters, 0, 3 * sizeof(unsigned long long), c->stream));
    launch_find_leavers(c->g, S.buf[S.cur], S.n, dim, side, out, cap, leaver_idx, counters, c->stream);
    c->launches += 1;
    unsigned long long L = 0;
    CU(c, cudaMemcpyAsync(&L, counters, sizeof(L), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    if ((long long)L > cap) {
        if (!remaining || cap == 0)
            return fail(c, PIC_ENOMEM, "%llu particles leave through this face, room for %lld (buffer, or np_max / 3)", L, cap);
        *remaining = (long long)L - cap;     // entries 0 .. cap-1 of the list are complete: take those out now
        L = (unsigned long long)cap;
    }
    *count = (long long)L;
    if (L > 0) {
        c->launches += launch_close_holes(S.buf[S.cur], S.n, (long long)L, leaver_idx, tailflag, fillers, counters, c->stream);
        S.n -= (long long)L;
        S.sorted = false;
        S.keys_valid = false;
        S.degraded = false;
    }
    CU(c, cudaGetLastError());
    return PIC_OK;
}

// Deletes every particle beyond face (dim, side), in batches of np_max / 3 (the size of the index scratch), so that
// a caller of pic_shift_window or of a step with absorbing faces never meets that limit half way through.
static int discard_leavers(pic_ctx* c, Species& S, int dim, int side, long long* count) {
    *count = 0;
    long long left = 0;
    do {
        long long got = 0;
        int rc = take_leavers(c, S, dim, side, nullptr, S.np_max / 3, &got, &left);
        if (rc != PIC_OK) return rc;
        *count += got;
        c->deleted += (unsigned long long)got;
    } while (left > 0);
    return PIC_OK;
}

static int discard_at_absorbing_faces(pic_ctx* c) {
    for (int d = 0; d < 3; ++d)
        if ((c->absorb_mask >> d) & 1)
            for (int s = 0; s < c->nspecies; ++s)
                for (int side = 0; side < 2; ++side) {
                    long long cnt;
                    int rc = discard_leavers(c, c->sp[s], d, side, &cnt);
                    if (rc != PIC_OK) return rc;
                }
    return PIC_OK;
}

// mask: bit 0 = J := 0, particles, J fold (and smoothing); bit 1 = first B half push; bit 2 = E push;
// bit 3 = second B half push (ends the step).  pic_step runs all four; pic_step_stage one at a time (bricks).
static int sort_impl(pic_ctx* c);

static int step_impl(pic_ctx* c, int nsteps, int mask) {
    if (nsteps < 0) return fail(c, PIC_EINVAL, "nsteps < 0");
    bool any = false;
    for (int s = 0; s < c->nspecies; ++s) any = any || c->sp[s].loaded;
    if (!any) return fail(c, PIC_ESTATE, "pic_step before any pic_load_particles");
    if (c->force_path == 2)
        for (int s = 0; s < c->nspecies; ++s)
            if (c->sp[s].loaded && !c->sp[s].sorted)
                return fail(c, PIC_ESTATE, "force_path=2 needs pic_sort before pic_step (species %d)", s);
    const bool timing = c->stage_timing != 0 && mask == 15;
    const Grid& g = c->g;
    const size_t comp_bytes = (size_t)g.npad * sizeof(double);
    const YeeMaps* tma_B = ((c->yee_tma & 1) && c->yee_tma_ok) ? &c->yee_maps : nullptr;
    const YeeMaps* tma_E = ((c->yee_tma & 2) && c->yee_tma_ok) ? &c->yee_maps : nullptr;
    for (int it = 0; it < nsteps; ++it) {
        if ((mask & 1) && c->auto_sort > 0) {
            // option "auto_sort" = k: the library keeps the fused per-tile kernel on its fast path by sorting (deferred:
            // keys, ranks and the permutation only) whenever a species is unsorted or has taken k steps since its last sort
            bool due = false;
            for (int s = 0; s < c->nspecies; ++s) {
                const Species& S = c->sp[s];
                due = due || (S.loaded && S.n > 0 && (!S.sorted || S.steps_since_sort >= c->auto_sort));
            }
            if (due) {
                const int rc = sort_impl(c);
                if (rc != PIC_OK) return rc;
            }
        }
        cudaEvent_t* ev = nullptr;
        if (timing) {
            size_t first;
            if (!take_events(c, EV_PER_STEP, &first)) return fail(c, PIC_ECUDA, "cudaEventCreate failed");
            c->spans.push_back(TimedSpan{first, 0});
            ev = c->ev_pool.data() + first;
            cudaEventRecord(ev[0], c->stream);
        }
        nvtxRangePushA("pic_step");
        if (mask & 1) {
        // J := 0 (R13).  Jx,Jy,Jz are contiguous in the arena.
        nvtxRangePushA("zero_J");
        if (c->f.Jx < c->f.Jy && c->f.Jy < c->f.Jz) {     // one memset over the three components (and the alignment gaps)
            CU(c, cudaMemsetAsync(c->f.Jx, 0, (size_t)((char*)c->f.Jz - (char*)c->f.Jx) + comp_bytes, c->stream));
        } else {
            CU(c, cudaMemsetAsync(c->f.Jx, 0, comp_bytes, c->stream));
            CU(c, cudaMemsetAsync(c->f.Jy, 0, comp_bytes, c->stream));
            CU(c, cudaMemsetAsync(c->f.Jz, 0, comp_bytes, c->stream));
        }
        nvtxRangePop();
        if (timing) cudaEventRecord(ev[1], c->stream);
        // steps 1-5 per species, in index order (R37)
        nvtxRangePushA("particles");
        if (c->drift_watch) poll_watch(c);
        // the watch is re-armed only when no earlier snapshot is still in flight (its pinned slots are reused)
        const bool watch = c->drift_watch && !c->watch_armed && c->force_path == 0;
        if (watch) {
            CU(c, cudaMemcpyAsync(&c->watch[0], c->status, sizeof(DevStatus), cudaMemcpyDeviceToHost, c->stream));
            for (int s = 0; s < c->nspecies; ++s) c->watch_tile[s] = false;
        }
        for (int s = 0; s < c->nspecies; ++s) {
            Species& S = c->sp[s];
            if (S.loaded && S.n > 0) {
                if (use_tile_path(c, S)) {
                    // a deferred sort is carried out here: inputs read through perm, outputs to the other buffer
                    const bool deferred = S.perm_pending;
                    const Particles& P = S.buf[S.cur];
                    const Particles& PO = deferred ? S.buf[S.cur ^ 1] : P;
                    const bool keys = c->fuse_keys != 0;
                    c->launches += launch_particles_tile(g, c->f, P, PO, deferred ? S.perm : nullptr,
                                                         keys ? S.key : nullptr, S.n, S.q, S.m, c->order, c->gather_variant,
                                                         c->precision, S.cell_offset,
                                                         S.steps_since_sort == 0 && c->tile_fresh != 0, c->status,
                                                         c->stream);
                    S.keys_valid = keys;
                    if (deferred) {
                        S.cur ^= 1;
                        S.perm_pending = false;
                    }
                    if (watch) c->watch_tile[s] = true;
                } else {
                    if (S.sorted && S.degraded) c->fallbacks += 1;
                    materialize(c, S);
                    S.keys_valid = false;
                    launch_particles_global(g, c->f, S.buf[S.cur], S.n, S.q, S.m, c->order, c->gather_variant,
                                            c->deposit_variant, c->precision, c->status, c->stream);
                    c->launches += 1;
                }
                S.steps_since_sort += 1;
            }
            if (watch)
                CU(c, cudaMemcpyAsync(&c->watch[s + 1], c->status, sizeof(DevStatus), cudaMemcpyDeviceToHost, c->stream));
        }
        if (watch) {
            CU(c, cudaEventRecord(c->watch_ev, c->stream));
            c->watch_armed = true;
            c->watch_sorts = c->sorts;
        }
        nvtxRangePop();
        if (timing) cudaEventRecord(ev[2], c->stream);
        // periodic fold of the J guard cells into the interior
        nvtxRangePushA("fold_J");
        launch_fold_guards3(g, c->f.Jx, c->f.Jy, c->f.Jz, c->stream);
        c->launches += 1;
        if (c->smooth_passes > 0) {      // NEXT-3: binomial smoothing of J before the E push
            double* J[3] = {c->f.Jx, c->f.Jy, c->f.Jz};
            for (int k = 0; k < 3; ++k) c->launches += launch_smooth_binomial(g, J[k], c->tmp, c->smooth_passes, c->stream);
        }
        nvtxRangePop();
        if (c->absorb_mask) {            // NEXT-2: whoever left through an open end is gone (synchronises)
            int rc = discard_at_absorbing_faces(c);
            if (rc != PIC_OK) { nvtxRangePop(); return rc; }
        }
        }      // mask & 1
        if (timing) cudaEventRecord(ev[3], c->stream);
        // steps 6-8
        nvtxRangePushA("yee");
        if (mask & 2) {
            launch_push_B(g, c->f, 0.5 * g.dt, tma_B, c->stream);
            c->launches += 1;
            if (c->absorb_mask) zero_absorbing_guards(c, 1);
            damp_layers(c, 1);
        }
        if (timing) cudaEventRecord(ev[4], c->stream);
        if (mask & 4) {
            launch_push_E(g, c->f, g.dt, tma_E, c->stream);
            c->launches += 1;
            if (c->absorb_mask) zero_absorbing_guards(c, 0);
            damp_layers(c, 0);
        }
        if (timing) cudaEventRecord(ev[5], c->stream);
        if (mask & 8) {
            launch_push_B(g, c->f, 0.5 * g.dt, tma_B, c->stream);
            c->launches += 1;
            if (c->absorb_mask) zero_absorbing_guards(c, 1);
            damp_layers(c, 1);
            c->steps += 1;
        }
        nvtxRangePop();
        if (timing) cudaEventRecord(ev[6], c->stream);
        nvtxRangePop();
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e, "pic_step launch");
    return PIC_OK;
}

int pic_step(pic_ctx* c, int nsteps) {
    ENTER(c);
    if (c->g.open_mask & ~c->absorb_mask)
        return fail(c, PIC_ESTATE, "a brick (open_mask != 0) is stepped with pic_step_stage and the halo calls");
    if (c->smooth_passes > 0 && c->g.open_mask) return fail(c, PIC_ESTATE, "smooth_passes is not available with open faces");
    return step_impl(c, nsteps, 15);
}

int pic_step_stage(pic_ctx* c, int stage) {
    ENTER(c);
    if (stage < 0 || stage > 3) return fail(c, PIC_EINVAL, "stage must be 0 .. 3");
    if (c->smooth_passes > 0 && c->g.open_mask) return fail(c, PIC_ESTATE, "smooth_passes is not available on a brick");
    if (stage == 0 && c->nspecies > 0) {
        bool any = false;
        for (int s = 0; s < c->nspecies; ++s) any = any || c->sp[s].loaded;
        if (!any) return fail(c, PIC_ESTATE, "pic_step_stage before any pic_load_particles");
    }
    return step_impl(c, 1, 1 << stage);
}

// ---- NEXT-1: what a brick hands to its neighbours (bricks.cu) ------------------------------------------
long long pic_halo_doubles(pic_ctx* c, int dim) {
    if (!c || dim < 0 || dim > 2) return -1;
    return 3 * halo_doubles(c->g, dim);
}

static int halo_args(pic_ctx* c, int group, int dim, int side, const void* buf) {
    if (group < 0 || group > 2 || dim < 0 || dim > 2 || side < 0 || side > 1 || !buf)
        return fail(c, PIC_EINVAL, "bad halo group, dim, side or buffer");
    const int n = (dim == 0) ? c->g.nx : ((dim == 1) ? c->g.ny : c->g.nz);
    if (n < NG) return fail(c, PIC_EINVAL, "a brick needs at least %d cells along an exchanged dimension", NG);
    return PIC_OK;
}

int pic_export_halo(pic_ctx* c, int group, int dim, int side, double* buf_dev) {
    ENTER(c);
    int rc = halo_args(c, group, dim, side, buf_dev);
    if (rc != PIC_OK) return rc;
    const Grid& g = c->g;
    double* F[3][3] = {{c->f.Ex, c->f.Ey, c->f.Ez}, {c->f.Bx, c->f.By, c->f.Bz}, {c->f.Jx, c->f.Jy, c->f.Jz}};
    const int n = (dim == 0) ? g.nx : ((dim == 1) ? g.ny : g.nz);
    // E, B: the interior layers next to the face; J: the guard layers beyond it
    const int first = (group == 2) ? (side ? n : -NG) : (side ? n - NG : 0);
    const long long per = halo_doubles(g, dim);
    for (int k = 0; k < 3; ++k) launch_halo_pack(g, F[group][k], dim, first, buf_dev + k * per, c->stream);
    c->launches += 3;
    CU(c, cudaGetLastError());
    return PIC_OK;
}

int pic_import_halo(pic_ctx* c, int group, int dim, int side, const double* buf_dev) {
    ENTER(c);
    int rc = halo_args(c, group, dim, side, buf_dev);
    if (rc != PIC_OK) return rc;
    const Grid& g = c->g;
    double* F[3][3] = {{c->f.Ex, c->f.Ey, c->f.Ez}, {c->f.Bx, c->f.By, c->f.Bz}, {c->f.Jx, c->f.Jy, c->f.Jz}};
    const int n = (dim == 0) ? g.nx : ((dim == 1) ? g.ny : g.nz);
    // E, B: into the guard layers beyond the face; J: ADDED to the interior layers next to it
    const int first = (group == 2) ? (side ? n - NG : 0) : (side ? n : -NG);
    const long long per = halo_doubles(g, dim);
    for (int k = 0; k < 3; ++k)
        launch_halo_unpack(g, F[group][k], dim, first, buf_dev + k * per, group == 2, c->stream);
    c->launches += 3;
    CU(c, cudaGetLastError());
    return PIC_OK;
}

int pic_export_leavers(pic_ctx* c, int species, int dim, int side, double* buf_dev, long long capacity,
                       long long* count) {
    ENTER(c);
    if (species < 0 || species >= c->nspecies || dim < 0 || dim > 2 || side < 0 || side > 1 || !count ||
        capacity < 0 || (capacity > 0 && !buf_dev))
        return fail(c, PIC_EINVAL, "bad argument of pic_export_leavers");
    Species& S = c->sp[species];
    return take_leavers(c, S, dim, side, buf_dev, capacity, count);
}

int pic_import_arrivals(pic_ctx* c, int species, const double* buf_dev, long long count, double shift_x, double shift_y,
                        double shift_z) {
    ENTER(c);
    if (species < 0 || species >= c->nspecies || count < 0 || (count > 0 && !buf_dev))
        return fail(c, PIC_EINVAL, "bad argument of pic_import_arrivals");
    Species& S = c->sp[species];
    if (!S.loaded) return fail(c, PIC_ESTATE, "species %d was never loaded (load it, empty if need be, to set q and m)", species);
    if (count == 0) return PIC_OK;
    if (S.n + count > S.np_max) return fail(c, PIC_ENOMEM, "%lld arrivals do not fit: n = %lld, np_max = %lld", count, S.n, S.np_max);
    materialize(c, S);
    launch_append_arrivals(S.buf[S.cur], S.n, buf_dev, count, shift_x, shift_y, shift_z, c->stream);
    c->launches += 1;
    S.n += count;
    S.sorted = false;
    S.keys_valid = false;
    CU(c, cudaGetLastError());
    return PIC_OK;
}

// ---- NEXT-2: moving window and plane source ----------------------------------------------------------------
int pic_shift_window(pic_ctx* c, int ncells, long long* deleted) {
    ENTER(c);
    if (!(c->absorb_mask & 4)) return fail(c, PIC_ESTATE, "a moving window needs open ends along z (absorb_mask bit 2)");
    if (ncells < 0 || ncells > c->g.nz) return fail(c, PIC_EINVAL, "ncells must be 0 .. nz");
    if (deleted) *deleted = 0;
    if (ncells == 0) return PIC_OK;
    double* F[9] = {c->f.Ex, c->f.Ey, c->f.Ez, c->f.Bx, c->f.By, c->f.Bz, c->f.Jx, c->f.Jy, c->f.Jz};
    for (int k = 0; k < 9; ++k) launch_shift_z(c->g, F[k], ncells, c->stream);
    c->launches += 9;
    // the planes that slid into the lower guard layers are outside the box now
    zero_absorbing_guards(c, 0);
    zero_absorbing_guards(c, 1);
    zero_absorbing_guards(c, 2);
    Grid& g = c->g;
    g.zmin += ncells * g.dz;           // the same expression the oracle uses (its zmin + n dz)
    g.zmax = g.zmin + g.Lz;
    long long total = 0;
    for (int s = 0; s < c->nspecies; ++s) {
        Species& S = c->sp[s];
        if (!S.loaded) continue;
        long long cnt = 0;
        int rc = discard_leavers(c, S, 2, 0, &cnt);
        if (rc != PIC_OK) return rc;
        total += cnt;
        S.sorted = false;              // every cell index changed
        S.keys_valid = false;
        S.perm_pending = false;
    }
    if (deleted) *deleted = total;
    CU(c, cudaGetLastError());
    return PIC_OK;
}

int pic_set_damping(pic_ctx* c, int ncells, const double* factors) {
    ENTER(c);
    if (ncells < 0 || ncells > DAMP_MAX || (ncells > 0 && !factors))
        return fail(c, PIC_EINVAL, "damping layer of 0 .. %d cells, factors given", DAMP_MAX);
    if (ncells > 0 && !(c->absorb_mask & 4))
        return fail(c, PIC_ESTATE, "damping layers sit in front of open z ends (absorb_mask bit 2)");
    if (2 * ncells > c->g.nz) return fail(c, PIC_EINVAL, "the two layers overlap (nz = %d)", c->g.nz);
    for (int m = 0; m < ncells; ++m)
        if (!std::isfinite(factors[m])) return fail(c, PIC_EINVAL, "factor %d is not finite", m);
    c->damp.n = ncells;
    for (int m = 0; m < ncells; ++m) c->damp.f[m] = factors[m];
    return PIC_OK;
}

int pic_add_plane(pic_ctx* c, int component, int k, const double* values, int src_on_device) {
    ENTER(c);
    if (component < 0 || component > 8 || k < 0 || k >= c->g.nz || !values)
        return fail(c, PIC_EINVAL, "bad component, plane or buffer");
    double* F[9] = {c->f.Ex, c->f.Ey, c->f.Ez, c->f.Bx, c->f.By, c->f.Bz, c->f.Jx, c->f.Jy, c->f.Jz};
    const double* src = values;
    if (!src_on_device) {
        CU(c, cudaMemcpyAsync(c->tmp, values, (size_t)c->g.nx * c->g.ny * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        src = c->tmp;
    }
    launch_add_plane(c->g, F[component], k, src, c->stream);
    c->launches += 1;
    CU(c, cudaGetLastError());
    if (!src_on_device) CU(c, cudaStreamSynchronize(c->stream));
    return PIC_OK;
}

int pic_sort(pic_ctx* c) {
    ENTER(c);
    bool any = false;
    for (int s = 0; s < c->nspecies; ++s) any = any || c->sp[s].loaded;
    if (!any) return fail(c, PIC_ESTATE, "pic_sort before any pic_load_particles");
    return sort_impl(c);
}

// every loaded species; asynchronous (pic_sort, and pic_step itself under the option "auto_sort")
static int sort_impl(pic_ctx* c) {
    cudaEvent_t* ev = nullptr;
    nvtxRangePushA("pic_sort");
    if (c->stage_timing) {
        size_t first;
        if (!take_events(c, EV_PER_SORT, &first)) { nvtxRangePop(); return fail(c, PIC_ECUDA, "cudaEventCreate failed"); }
        c->spans.push_back(TimedSpan{first, 1});
        ev = c->ev_pool.data() + first;
        cudaEventRecord(ev[0], c->stream);
    }
    for (int s = 0; s < c->nspecies; ++s) {
        Species& S = c->sp[s];
        if (!S.loaded) continue;
        // (a still pending deferred sort is simply superseded: the keys are taken from the unsorted buffer)
        const bool deferred = c->sort_deferred != 0 && c->force_path != 1;
        c->launches += launch_sort(c->g, S.buf[S.cur], S.buf[S.cur ^ 1], S.n, S.cell_offset,
                                   deferred ? S.perm : nullptr, S.keys_valid ? S.key : nullptr, c->sort_scratch,
                                   c->stream);
        S.keys_valid = false;
        if (deferred) S.perm_pending = S.n > 0;
        else { S.cur ^= 1; S.perm_pending = false; }
        S.sorted = true;
        S.steps_since_sort = 0;
        S.degraded = false;
    }
    if (ev) cudaEventRecord(ev[1], c->stream);
    nvtxRangePop();
    c->sorts += 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e, "pic_sort launch");
    return PIC_OK;
}

int pic_get_fields(pic_ctx* c, double* Ex, double* Ey, double* Ez, double* Bx, double* By, double* Bz, double* Jx,
                   double* Jy, double* Jz, int dst_on_device) {
    ENTER(c);
    double* dst[9] = {Ex, Ey, Ez, Bx, By, Bz, Jx, Jy, Jz};
    const double* src[9] = {c->f.Ex, c->f.Ey, c->f.Ez, c->f.Bx, c->f.By, c->f.Bz, c->f.Jx, c->f.Jy, c->f.Jz};
    for (int k = 0; k < 9; ++k) {
        int rc = copy_out(c, src[k], dst[k], dst_on_device);
        if (rc != PIC_OK) return rc;
    }
    return sync_and_check(c);
}

int pic_get_particles(pic_ctx* c, int species, long long* n, double* x, double* y, double* z, double* ux,
                      double* uy, double* uz, double* w, unsigned long long* id, int dst_on_device) {
    ENTER(c);
    if (species < 0 || species >= c->nspecies) return fail(c, PIC_EINVAL, "species index %d out of range", species);
    Species& S = c->sp[species];
    if (!S.loaded) return fail(c, PIC_ESTATE, "species %d was never loaded", species);
    if (n) *n = S.n;
    materialize(c, S);
    const Particles& P = S.buf[S.cur];
    const cudaMemcpyKind kind = dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    void* dst[8] = {x, y, z, ux, uy, uz, w, id};
    const void* src[8] = {P.x, P.y, P.z, P.ux, P.uy, P.uz, P.w, P.id};
    for (int a = 0; a < 8; ++a)
        if (dst[a] && S.n > 0) CU(c, cudaMemcpyAsync(dst[a], src[a], (size_t)S.n * 8, kind, c->stream));
    return sync_and_check(c);
}

int pic_deposit_rho(pic_ctx* c, int species, double* rho, int dst_on_device) {
    ENTER(c);
    if (species < -1 || species >= c->nspecies || !rho) return fail(c, PIC_EINVAL, "bad species index or NULL rho");
    if (species >= 0 && !c->sp[species].loaded) return fail(c, PIC_ESTATE, "species %d was never loaded", species);
    // tmp serves as the padded rho: deposit with global atomics, fold the guards, strip them on the way out
    CU(c, cudaMemsetAsync(c->tmp, 0, (size_t)c->g.npad * sizeof(double), c->stream));
    for (int s = 0; s < c->nspecies; ++s) {
        Species& S = c->sp[s];
        if (!S.loaded || (species >= 0 && s != species) || S.n == 0) continue;
        launch_deposit_rho(c->g, S.buf[S.cur], S.n, S.q, c->order, c->tmp, c->stream);
        c->launches += 1;
    }
    launch_fold_guards(c->g, c->tmp, c->stream);
    c->launches += 1;
    if (dst_on_device) {
        pack_kernel<<<cell_grid(c->g), 128, 0, c->stream>>>(c->g, c->tmp, rho);
        c->launches += 1;
    } else {
        // strided copy straight from the padded scratch to the caller's guard-free host array
        cudaMemcpy3DParms p;
        memset(&p, 0, sizeof(p));
        p.srcPtr = make_cudaPitchedPtr(c->tmp, (size_t)c->g.px * sizeof(double), (size_t)c->g.px, (size_t)c->g.py);
        p.srcPos = make_cudaPos((size_t)NG * sizeof(double), NG, NG);
        p.dstPtr = make_cudaPitchedPtr(rho, (size_t)c->g.nx * sizeof(double), (size_t)c->g.nx, (size_t)c->g.ny);
        p.extent = make_cudaExtent((size_t)c->g.nx * sizeof(double), (size_t)c->g.ny, (size_t)c->g.nz);
        p.kind = cudaMemcpyDeviceToHost;
        CU(c, cudaMemcpy3DAsync(&p, c->stream));
    }
    return sync_and_check(c);
}

int pic_get_cell_offsets(pic_ctx* c, int species, unsigned int* offsets, int dst_on_device) {
    ENTER(c);
    if (species < 0 || species >= c->nspecies || !offsets) return fail(c, PIC_EINVAL, "bad species or NULL offsets");
    Species& S = c->sp[species];
    if (!S.loaded || !S.sorted) return fail(c, PIC_ESTATE, "species %d was never sorted", species);
    const size_t bytes = ((size_t)c->g.nx * c->g.ny * c->g.nz + 1) * sizeof(unsigned int);
    CU(c, cudaMemcpyAsync(offsets, S.cell_offset, bytes,
                          dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
    return sync_and_check(c);
}

int pic_get_counters(pic_ctx* c, unsigned long long* counters) {
    if (!counters) return PIC_EINVAL;
    ENTER(c);
    DevStatus h;
    CU(c, cudaMemcpyAsync(&h, c->status, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    counters[0] = h.n_fast;
    counters[1] = h.n_slow;
    counters[2] = h.n_global;
    counters[3] = c->launches;
    counters[4] = c->steps;
    counters[5] = c->sorts;
    counters[6] = c->yee_tma_ok ? 1ull : 0ull;
    counters[7] = c->fallbacks;
    counters[8] = c->deleted;
    return PIC_OK;
}

int pic_get_stage_ms(pic_ctx* c, float* ms) {
    ENTER(c);
    if (!ms) return PIC_EINVAL;
    if (!c->stage_timing) return fail(c, PIC_ESTATE, "stage timing is off");
    CU(c, cudaStreamSynchronize(c->stream));
    for (int k = 0; k < NSTAGE; ++k) ms[k] = 0.f;
    for (const TimedSpan& sp : c->spans) {
        const cudaEvent_t* ev = c->ev_pool.data() + sp.first;
        float t = 0.f;
        if (sp.kind == 0) {
            // spans between the 7 events: zero J, particles, fold, B half, E, B half
            static const int stage_of[6] = {0, 1, 2, 3, 4, 3};
            for (int k = 0; k < 6; ++k) {
                CU(c, cudaEventElapsedTime(&t, ev[k], ev[k + 1]));
                ms[stage_of[k]] += t;
            }
            ms[6] += 1.f;
        } else {
            CU(c, cudaEventElapsedTime(&t, ev[0], ev[1]));
            ms[5] += t;
            ms[7] += 1.f;
        }
    }
    c->spans.clear();
    c->ev_used = 0;
    return PIC_OK;
}

int pic_set_option(pic_ctx* c, const char* name, long long value) {
    ENTER(c);
    if (!name) return PIC_EINVAL;
    if (!strcmp(name, "stage_timing")) {
        if (cudaStreamSynchronize(c->stream) != cudaSuccess) return fail(c, PIC_ECUDA, "cudaStreamSynchronize");
        c->stage_timing = value != 0;
        c->spans.clear();
        c->ev_used = 0;
    }
    else if (!strcmp(name, "force_path")) {
        if (value < 0 || value > 2) return fail(c, PIC_EINVAL, "force_path must be 0, 1 or 2");
        c->force_path = (int)value;
    } else if (!strcmp(name, "yee_tma")) c->yee_tma = (int)value & 3;
    else if (!strcmp(name, "tile_fresh")) c->tile_fresh = value != 0;
    else if (!strcmp(name, "sort_deferred")) c->sort_deferred = value != 0;
    else if (!strcmp(name, "fuse_keys")) c->fuse_keys = value != 0;
    else if (!strcmp(name, "drift_watch")) c->drift_watch = value != 0;
    else if (!strcmp(name, "auto_sort")) {
        if (value < 0 || value > 1000000) return fail(c, PIC_EINVAL, "auto_sort must be 0 (off) or a number of steps");
        c->auto_sort = (int)value;
    }
    else if (!strcmp(name, "open_mask")) {
        if (value < 0 || value > 7) return fail(c, PIC_EINVAL, "open_mask must be 0 .. 7");
        c->g.open_mask = (int)value | c->absorb_mask;     // an absorbing face stays open whatever the brick layout says
    } else if (!strcmp(name, "absorb_mask")) {
        if (value < 0 || value > 7) return fail(c, PIC_EINVAL, "absorb_mask must be 0 .. 7");
        const int n[3] = {c->g.nx, c->g.ny, c->g.nz};
        for (int d = 0; d < 3; ++d)
            if (((value >> d) & 1) && n[d] < NG) return fail(c, PIC_EINVAL, "an open end needs at least %d cells along its dimension", NG);
        c->g.open_mask = (c->g.open_mask & ~c->absorb_mask) | (int)value;
        c->absorb_mask = (int)value;
        if (!(value & 4)) c->damp.n = 0;            // the layers go with the open z ends
        zero_absorbing_guards(c, 0);
        zero_absorbing_guards(c, 1);
        CU(c, cudaGetLastError());
    } else if (!strcmp(name, "id_base")) {
        if (value < 0) return fail(c, PIC_EINVAL, "id_base must be >= 0");
        c->id_base = (unsigned long long)value;
    } else if (!strcmp(name, "gather_variant")) {
        if (value < 0 || value > 1) return fail(c, PIC_EINVAL, "gather_variant must be 0 or 1");
        c->gather_variant = (int)value;
    } else if (!strcmp(name, "precision")) {
        if (value < 0 || value > 1) return fail(c, PIC_EINVAL, "precision must be 0 (fp64) or 1 (fp32 fields and momenta)");
        c->precision = (int)value;
    } else if (!strcmp(name, "deposit_variant")) {
        if (value < 0 || value > 1) return fail(c, PIC_EINVAL, "deposit_variant must be 0 or 1");
        if (value && c->force_path == 2) return fail(c, PIC_ESTATE, "direct deposition runs in the global-atomic kernel: not with force_path = 2");
        c->deposit_variant = (int)value;
    } else if (!strcmp(name, "smooth_passes")) {
        if (value < 0 || value > 16) return fail(c, PIC_EINVAL, "smooth_passes must be 0 .. 16");
        c->smooth_passes = (int)value;
    }
    else return fail(c, PIC_EINVAL, "unknown option '%s'", name);
    return PIC_OK;
}

int pic_sync(pic_ctx* c) {
    ENTER(c);
    return sync_and_check(c);
}

const char* pic_last_error(pic_ctx* c) {
    if (!c) return "NULL context";
    return c->err;
}

int pic_destroy(pic_ctx* c) {
    if (!c) return PIC_EINVAL;
    cudaSetDevice(c->device);
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    if (c->watch_ev) {
        cudaEventSynchronize(c->watch_ev);      // a snapshot copy may still be writing the pinned block
        cudaEventDestroy(c->watch_ev);
    }
    if (c->watch) cudaFreeHost(c->watch);
    delete c;
    return PIC_OK;
}

}  // extern "C"
