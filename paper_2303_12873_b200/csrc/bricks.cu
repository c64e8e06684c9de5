// bricks.cu -- what one brick of a domain decomposition exchanges with its neighbours (SURVEY.md 8(e) and
// 8(f) NEXT-1; the paper's weak scaling rests on a spatial decomposition with neighbour
// exchange).  Each brick is an ordinary context of this library whose grid is its own block of cells; along a
// decomposed dimension (Grid::open_mask) the brick's guard layers stand for the neighbour's cells instead of
// periodic images of its own:
//   E, B   the NG interior layers next to a face go to the neighbour's guard layers (copy)
//   J      the NG guard layers beyond a face go to the neighbour's interior layers (sum)
//   particles that left through a face travel as 8-double records and are appended to the neighbour's container
// The kernels here only pack, unpack and partition; who talks to whom is the caller's schedule
// (paper_2303_12873_b200/bricks.py), over NCCL send/recv, peer copies, or plain pointers on one GPU.
#include "pic_internal.h"

namespace pic {

namespace {

// extents of the plane spanned by the two dimensions other than `dim` (padded), and strides of all three
struct PlaneGeom {
    int n1, n2;              // padded extents of the two in-plane dimensions (lower dimension first)
    long long s0, s1, s2;    // strides: along dim, along the two in-plane dimensions
};

__host__ __device__ inline PlaneGeom plane_geom(const Grid& g, int dim) {
    PlaneGeom p;
    const int ext[3] = {g.nx + 2 * NG, g.py, g.pz};
    const long long str[3] = {1, g.sy, g.sz};
    const int d1 = (dim == 0) ? 1 : 0, d2 = (dim == 2) ? 1 : 2;
    p.n1 = ext[d1]; p.n2 = ext[d2];
    p.s0 = str[dim]; p.s1 = str[d1]; p.s2 = str[d2];
    return p;
}

// buf[l][v][u] <-> F at layer first_layer + l along dim (interior index, may be negative), in-plane padded (u, v)
template <bool PACK, bool ADD>
__global__ void halo_kernel(Grid g, PlaneGeom pg, double* F, int dim, int first_layer, double* buf) {
    const int u = (int)(blockIdx.x * blockDim.x + threadIdx.x), v = (int)blockIdx.y, l = (int)blockIdx.z;
    if (u >= pg.n1) return;
    const long long o = pg.s0 * (long long)(first_layer + l + NG) + pg.s1 * u + pg.s2 * v;
    const long long b = ((long long)l * pg.n2 + v) * pg.n1 + u;
    if (PACK) buf[b] = F[o];
    else if (ADD) F[o] += buf[b];
    else F[o] = buf[b];
}

// every layer first_layer .. first_layer + NG - 1 along dim := value (full padded extent of the other two dimensions)
__global__ void halo_fill_kernel(PlaneGeom pg, double* F, int first_layer, double value) {
    const int u = (int)(blockIdx.x * blockDim.x + threadIdx.x), v = (int)blockIdx.y, l = (int)blockIdx.z;
    if (u >= pg.n1) return;
    F[pg.s0 * (long long)(first_layer + l + NG) + pg.s1 * u + pg.s2 * v] = value;
}

// moving window: F[k] := F[k + n] along z over the whole padded array, zero where k + n runs off the top.  One thread
// per (x, y) column walks z upwards, so every read happens before the write that would overwrite it.
__global__ void shift_z_kernel(Grid g, double* F, int n) {
    const int i = (int)(blockIdx.x * blockDim.x + threadIdx.x), j = (int)blockIdx.y;
    if (i >= g.px) return;
    double* col = F + i + g.sy * j;
    for (int k = 0; k < g.pz; ++k) col[g.sz * k] = (k + n < g.pz) ? col[g.sz * (k + n)] : 0.0;
}

// F[interior plane k] += values (guard-free nx x ny, x fastest)
__global__ void add_plane_kernel(Grid g, double* F, int k, const double* __restrict__ values) {
    const int i = (int)(blockIdx.x * blockDim.x + threadIdx.x), j = (int)blockIdx.y;
    if (i < g.nx) F[g.idx(i, j, k)] += values[i + (long long)g.nx * j];
}

// damping layers in front of the two open z ends: plane m cells from a face (m = 0 next to it) *= t.f[m], over the
// whole padded x-y extent (the x / y guard cells hold periodic images of the same plane), three components at once
__global__ void damp_z_kernel(Grid g, double* F0, double* F1, double* F2, DampTable t) {
    const int i = (int)(blockIdx.x * blockDim.x + threadIdx.x), j = (int)blockIdx.y;
    if (i >= g.px) return;
    const int m = (int)blockIdx.z >> 1, k = (blockIdx.z & 1) ? g.nz - 1 - m : m;
    const long long at = i + g.sy * j + g.sz * (long long)(k + NG);
    const double fm = t.f[m];
    F0[at] *= fm;
    F1[at] *= fm;
    F2[at] *= fm;
}

// ---- leavers: taken out of the container IN PLACE ------------------------------------------------------------
// Only a sliver of a brick's particles leaves through a face in one step, so the container is not copied: pass 1
// reads ONE coordinate of every particle, appends the index of every leaver to a list and its record to the
// message (8 B per particle instead of 128); the holes the leavers leave below the new end n' = n - L are then
// filled with the stayers found among the last L places (lists of L entries).  The order of the container
// changes: the species counts as unsorted afterwards.
__global__ void find_leavers_kernel(Grid g, Particles p, long long n, int dim, int side, double* out, long long capacity,
                                    unsigned int* leaver_idx, unsigned long long* counters) {
    const long long ip = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    bool leaves = false;
    if (ip < n) {
        const double pos = (dim == 0) ? p.x[ip] : ((dim == 1) ? p.y[ip] : p.z[ip]);
        const double lo = (dim == 0) ? g.xmin : ((dim == 1) ? g.ymin : g.zmin);
        const double hi = (dim == 0) ? g.xmax : ((dim == 1) ? g.ymax : g.zmax);
        leaves = side ? (pos >= hi) : (pos < lo);
    }
    const unsigned active = __activemask();
    const unsigned m = __ballot_sync(active, leaves);
    if (!m) return;
    const int leader = __ffs(active) - 1;
    unsigned long long base = 0;
    if (lane == leader) base = atomicAdd(&counters[0], (unsigned long long)__popc(m));
    base = __shfl_sync(active, base, leader);
    if (leaves) {
        const long long k = (long long)base + __popc(m & ((1u << lane) - 1u));
        if (k < capacity) {
            leaver_idx[k] = (unsigned int)ip;
            if (out) {
                double* r = out + 8 * k;
                r[0] = p.x[ip]; r[1] = p.y[ip]; r[2] = p.z[ip]; r[3] = p.ux[ip]; r[4] = p.uy[ip]; r[5] = p.uz[ip];
                r[6] = p.w[ip];
                r[7] = __longlong_as_double((long long)p.id[ip]);
            }
        }
    }
}

// tailflag[j] = 1 if place n' + j holds a leaver
__global__ void mark_tail_kernel(const unsigned int* leaver_idx, long long L, long long nprime, unsigned int* tailflag) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < L && (long long)leaver_idx[k] >= nprime) tailflag[(long long)leaver_idx[k] - nprime] = 1u;
}

// fillers = the stayers among the last L places
__global__ void list_fillers_kernel(const unsigned int* tailflag, long long L, long long nprime, unsigned int* fillers,
                                    unsigned long long* counters) {
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j < L && !tailflag[j]) fillers[atomicAdd(&counters[1], 1ull)] = (unsigned int)(nprime + j);
}

// every hole below n' receives one filler
__global__ void fill_holes_kernel(Particles p, const unsigned int* leaver_idx, long long L, long long nprime,
                                  const unsigned int* fillers, unsigned long long* counters) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= L) return;
    const long long hole = leaver_idx[k];
    if (hole >= nprime) return;
    const long long src = fillers[atomicAdd(&counters[2], 1ull)];
    p.x[hole] = p.x[src]; p.y[hole] = p.y[src]; p.z[hole] = p.z[src];
    p.ux[hole] = p.ux[src]; p.uy[hole] = p.uy[src]; p.uz[hole] = p.uz[src];
    p.w[hole] = p.w[src];
    p.id[hole] = p.id[src];
}

__global__ void append_arrivals_kernel(Particles dst, long long at, const double* in, long long count, double sx,
                                       double sy, double sz) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= count) return;
    const double* r = in + 8 * k;
    dst.x[at + k] = r[0] + sx; dst.y[at + k] = r[1] + sy; dst.z[at + k] = r[2] + sz;
    dst.ux[at + k] = r[3]; dst.uy[at + k] = r[4]; dst.uz[at + k] = r[5];
    dst.w[at + k] = r[6];
    dst.id[at + k] = (unsigned long long)__double_as_longlong(r[7]);
}

}  // namespace

long long halo_doubles(const Grid& g, int dim) {
    const PlaneGeom pg = plane_geom(g, dim);
    return (long long)NG * pg.n1 * pg.n2;
}

void launch_halo_pack(const Grid& g, const double* F, int dim, int first_layer, double* buf, cudaStream_t st) {
    const PlaneGeom pg = plane_geom(g, dim);
    dim3 bs(128, 1, 1), nb((pg.n1 + 127) / 128, pg.n2, NG);
    halo_kernel<true, false><<<nb, bs, 0, st>>>(g, pg, const_cast<double*>(F), dim, first_layer, buf);
}

void launch_halo_unpack(const Grid& g, double* F, int dim, int first_layer, const double* buf, bool add, cudaStream_t st) {
    const PlaneGeom pg = plane_geom(g, dim);
    dim3 bs(128, 1, 1), nb((pg.n1 + 127) / 128, pg.n2, NG);
    if (add) halo_kernel<false, true><<<nb, bs, 0, st>>>(g, pg, F, dim, first_layer, const_cast<double*>(buf));
    else halo_kernel<false, false><<<nb, bs, 0, st>>>(g, pg, F, dim, first_layer, const_cast<double*>(buf));
}

void launch_halo_fill(const Grid& g, double* F, int dim, int first_layer, double value, cudaStream_t st) {
    const PlaneGeom pg = plane_geom(g, dim);
    dim3 bs(128, 1, 1), nb((pg.n1 + 127) / 128, pg.n2, NG);
    halo_fill_kernel<<<nb, bs, 0, st>>>(pg, F, first_layer, value);
}

void launch_shift_z(const Grid& g, double* F, int ncells, cudaStream_t st) {
    dim3 bs(128, 1, 1), nb((g.px + 127) / 128, g.py, 1);
    shift_z_kernel<<<nb, bs, 0, st>>>(g, F, ncells);
}

void launch_add_plane(const Grid& g, double* F, int k, const double* values_dev, cudaStream_t st) {
    dim3 bs(128, 1, 1), nb((g.nx + 127) / 128, g.ny, 1);
    add_plane_kernel<<<nb, bs, 0, st>>>(g, F, k, values_dev);
}

void launch_damp_z(const Grid& g, double* F0, double* F1, double* F2, const DampTable& t, cudaStream_t st) {
    dim3 bs(128, 1, 1), nb((g.px + 127) / 128, g.py, 2 * t.n);
    damp_z_kernel<<<nb, bs, 0, st>>>(g, F0, F1, F2, t);
}

void launch_find_leavers(const Grid& g, const Particles& p, long long n, int dim, int side, double* out,
                         long long capacity, unsigned int* leaver_idx, unsigned long long* counters, cudaStream_t st) {
    if (n <= 0) return;
    find_leavers_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(g, p, n, dim, side, out, capacity, leaver_idx, counters);
}

int launch_close_holes(const Particles& p, long long n, long long L, const unsigned int* leaver_idx, unsigned int* tailflag,
                       unsigned int* fillers, unsigned long long* counters, cudaStream_t st) {
    if (L <= 0) return 0;
    const long long nprime = n - L;
    const unsigned nb = (unsigned)((L + 255) / 256);
    cudaMemsetAsync(tailflag, 0, (size_t)L * sizeof(unsigned int), st);
    mark_tail_kernel<<<nb, 256, 0, st>>>(leaver_idx, L, nprime, tailflag);
    list_fillers_kernel<<<nb, 256, 0, st>>>(tailflag, L, nprime, fillers, counters);
    fill_holes_kernel<<<nb, 256, 0, st>>>(p, leaver_idx, L, nprime, fillers, counters);
    return 3;
}

void launch_append_arrivals(const Particles& dst, long long at, const double* in, long long count, double sx, double sy,
                            double sz, cudaStream_t st) {
    if (count <= 0) return;
    append_arrivals_kernel<<<(unsigned)((count + 255) / 256), 256, 0, st>>>(dst, at, in, count, sx, sy, sz);
}

}  // namespace pic
