// particles_tile.cu -- fused gather + Boris push + Esirkepov deposition per
// cell-sorted tile (BASELINE.json:north_star parts
// 1-3, "fused per cell-sorted tile").
//
// One thread block owns a tile of TX x TY x TZ cells and the particles the last
// pic_sort listed in those cells (TY*TZ contiguous segments of the SoA arrays).
//   load    the tile's E,B stencil (+ halo for the shape support and D cells of
//           drift since the last sort) goes to shared memory; the J tile is zeroed
//   phase A particle-major, coalesced: thread <-> particle in container order.
//           Gather from the shared stencil (lanes of a warp sit in the same few
//           cells: broadcast LDS), Boris, move, coalesced store of the wrapped
//           state; (xi0,xi1,q*w) goes to a shared staging buffer.
//   phase B cell-major: lane <-> cell, so the 32 lanes of a warp deposit into 32
//           DIFFERENT windows and every shared-memory add of a warp instruction
//           hits 32 distinct addresses.  (fp64 atomicAdd on shared memory is a
//           CAS loop on sm_100a -- ATOMS.CAST.SPIN -- which costs 8.5 clk per warp
//           op with distinct addresses but 58 clk when 8 lanes share one; the
//           particle-major mapping of a sorted species would be the second case.)
//   flush   one global fp64 atomic (REDG.E.ADD.F64) per non-zero tile point.
// A particle whose cell left the tile's halo (drift > D cells, periodic wrap far
// from the tile) takes the global-memory update of particle_update.cuh instead:
// the kernel is correct for any particle order, only slower.
#include "particle_update.cuh"

namespace pic {

namespace {

constexpr int DRIFT = 1;   // cells a particle may sit outside its listed cell and still use the tile

template <int TX_, int TY_, int TZ_, int NT_, int CH_>
struct TileCfg {
    static constexpr int TX = TX_, TY = TY_, TZ = TZ_, NT = NT_, CH = CH_;
    static constexpr int NCELL = TX * TY * TZ;
    static constexpr int NSEG = TY * TZ;
    static constexpr int NSUB = NT / NCELL;               // threads per cell in phase B
    // gather stencil: nodes i-2 .. i+2 of a particle in cell i (every order, every staggering)
    static constexpr int GL = 2 + DRIFT;
    static constexpr int EX = TX + 2 * GL, EY = TY + 2 * GL, EZ = TZ + 2 * GL;
    static constexpr int ESZ = EX * EY * EZ;
    // deposit window: nodes i-2 .. i+3
    static constexpr int JL = 2 + DRIFT, JH = 3 + DRIFT;
    static constexpr int JX = TX + JL + JH + 1, JY = TY + JL + JH, JZ = TZ + JL + JH;   // JX even
    static constexpr int JSZ = JX * JY * JZ;
    static constexpr int STG = CH + CH / 8 + 8;           // skewed staging rows (slot + slot/8)
    static constexpr size_t SMEM = sizeof(double) * (6 * (size_t)ESZ + 3 * (size_t)JSZ + 7 * (size_t)STG) +
                                   sizeof(int) * (2 * NSEG + 2 + 2 * NCELL);
    static_assert(NT % NCELL == 0 && NSUB >= 1, "block size must be a multiple of the tile's cell count");
    static_assert(NCELL % 32 == 0, "a warp must map onto whole cells");
};

// Old and new nodal shapes on the common window of N+2 slots anchored at
// min(first old node, first new node); returns that node.  |move| < 1 cell.
template <int N>
__device__ __forceinline__ int shapes_pair(double xi0, double xi1, double (&s0)[N + 2], double (&ds)[N + 2],
                                           bool& bad) {
    double w0[N + 1], w1[N + 1];
    const int f0 = shape_weights<N>(xi0, w0);
    const int f1 = shape_weights<N>(xi1, w1);
    int s = f1 - f0;
    if (s < -1 || s > 1 || !(fabs(xi1 - xi0) < 1.0)) {
        bad = true;
        s = 0;
    }
#pragma unroll
    for (int a = 0; a < N + 2; ++a) {
        const double o_lo = (a >= 1) ? w0[a - 1] : 0.0;          // s < 0: old weight k sits in slot k+1
        const double o_eq = (a <= N) ? w0[(a <= N) ? a : 0] : 0.0;
        const double n_lo = (a >= 1) ? w1[a - 1] : 0.0;          // s > 0: new weight k sits in slot k+1
        const double n_eq = (a <= N) ? w1[(a <= N) ? a : 0] : 0.0;
        const double o = (s < 0) ? o_lo : o_eq;
        const double n = (s > 0) ? n_lo : n_eq;
        s0[a] = o;
        ds[a] = n - o;
    }
    return (s < 0) ? f1 : f0;
}

// Shared-memory adder: CAS-loop fp64 add (correct under any collision).
template <class C>
struct SmemAdder {
    double* J;    // 3 * JSZ
    __device__ __forceinline__ void operator()(int comp, int o, double v) const { atomicAdd(J + comp * C::JSZ + o, v); }
};

// Esirkepov deposition of one particle into the shared J tile.  (ox,oy,oz) =
// tile-relative slot of the window's first node.
template <int N, class C>
__device__ __forceinline__ void deposit_tile(double* Jt, int ox, int oy, int oz, const double (&s0x)[N + 2],
                                             const double (&dsx)[N + 2], const double (&s0y)[N + 2],
                                             const double (&dsy)[N + 2], const double (&s0z)[N + 2],
                                             const double (&dsz)[N + 2], double cx, double cy, double cz) {
    constexpr int W = N + 2;
    const int o0 = ox + C::JX * (oy + C::JY * oz);
    SmemAdder<C> add{Jt};
    {   // Jx[a,b,c] = cx * prefix_a(DSx) * (S0z[c] (S0y[b] + DSy[b]/2) + DSz[c] (S0y[b]/2 + DSy[b]/3))
        double pd[W - 1];
        double acc = 0.0;
#pragma unroll
        for (int a = 0; a < W - 1; ++a) { acc += dsx[a]; pd[a] = cx * acc; }
#pragma unroll
        for (int c = 0; c < W; ++c)
#pragma unroll
            for (int b = 0; b < W; ++b) {
                const double t = s0z[c] * (s0y[b] + 0.5 * dsy[b]) + dsz[c] * (0.5 * s0y[b] + (1.0 / 3.0) * dsy[b]);
                if (t != 0.0) {
#pragma unroll
                    for (int a = 0; a < W - 1; ++a) {
                        const double v = pd[a] * t;
                        if (v != 0.0) add(0, o0 + a + C::JX * (b + C::JY * c), v);
                    }
                }
            }
    }
    {   // Jy
        double pd[W - 1];
        double acc = 0.0;
#pragma unroll
        for (int b = 0; b < W - 1; ++b) { acc += dsy[b]; pd[b] = cy * acc; }
#pragma unroll
        for (int c = 0; c < W; ++c)
#pragma unroll
            for (int a = 0; a < W; ++a) {
                const double t = s0x[a] * (s0z[c] + 0.5 * dsz[c]) + dsx[a] * (0.5 * s0z[c] + (1.0 / 3.0) * dsz[c]);
                if (t != 0.0) {
#pragma unroll
                    for (int b = 0; b < W - 1; ++b) {
                        const double v = pd[b] * t;
                        if (v != 0.0) add(1, o0 + a + C::JX * (b + C::JY * c), v);
                    }
                }
            }
    }
    {   // Jz
        double pd[W - 1];
        double acc = 0.0;
#pragma unroll
        for (int c = 0; c < W - 1; ++c) { acc += dsz[c]; pd[c] = cz * acc; }
#pragma unroll
        for (int b = 0; b < W; ++b)
#pragma unroll
            for (int a = 0; a < W; ++a) {
                const double t = s0y[b] * (s0x[a] + 0.5 * dsx[a]) + dsy[b] * (0.5 * s0x[a] + (1.0 / 3.0) * dsx[a]);
                if (t != 0.0) {
#pragma unroll
                    for (int c = 0; c < W - 1; ++c) {
                        const double v = pd[c] * t;
                        if (v != 0.0) add(2, o0 + a + C::JX * (b + C::JY * c), v);
                    }
                }
            }
    }
}

// One component from the shared stencil; (fx,fy,fz) = tile slot of the first node.
template <int N, class C>
__device__ __forceinline__ double gather_tile(const double* __restrict__ F, int fx, int fy, int fz,
                                              const double (&wx)[N + 1], const double (&wy)[N + 1],
                                              const double (&wz)[N + 1]) {
    const double* base = F + fx + C::EX * (fy + C::EY * fz);
    double acc = 0.0;
#pragma unroll
    for (int c = 0; c <= N; ++c) {
        double accy = 0.0;
#pragma unroll
        for (int b = 0; b <= N; ++b) {
            const double* row = base + C::EX * (b + C::EY * c);
            double accx = 0.0;
#pragma unroll
            for (int a = 0; a <= N; ++a) accx = fma(wx[a], row[a], accx);
            accy = fma(wy[b], accx, accy);
        }
        acc = fma(wz[c], accy, acc);
    }
    return acc;
}

// tile-relative cell index with the periodic image nearest to the tile
__device__ __forceinline__ int rel_cell(int i, int t0, int T, int n) {
    int r = i - t0;
    if (r < -DRIFT) r += n;
    else if (r > T - 1 + DRIFT) r -= n;
    return r;
}

}  // namespace

namespace {

template <int N, class C>
__global__ void __launch_bounds__(C::NT, 1)
particles_tile_kernel(Grid g, Fields f, Particles p, double q, double h, const unsigned int* __restrict__ cell_offset,
                      int ntx, int nty, DevStatus* status) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* Et = reinterpret_cast<double*>(smem_raw);            // 6 * ESZ: Ex Ey Ez Bx By Bz
    double* Jt = Et + 6 * C::ESZ;                                // 3 * JSZ
    double* stg = Jt + 3 * C::JSZ;                               // 7 * STG
    int* seg_start = reinterpret_cast<int*>(stg + 7 * C::STG);   // NSEG: container index of the segment's first particle
    int* seg_pref = seg_start + C::NSEG;                         // NSEG + 1: tile index of the segment's first particle
    int* cell_lo = seg_pref + C::NSEG + 2;                       // NCELL: tile-index range of every cell
    int* cell_hi = cell_lo + C::NCELL;

    const int tid = threadIdx.x;
    int b = blockIdx.x;
    const int bx = b % ntx; b /= ntx;
    const int by = b % nty;
    const int bz = b / nty;
    const int t0x = bx * C::TX, t0y = by * C::TY, t0z = bz * C::TZ;

    // ---- segments and cell ranges -------------------------------------------------
    if (tid < C::NSEG) {
        const int j = t0y + tid % C::TY, k = t0z + tid / C::TY;
        int s0 = 0, len = 0;
        if (j < g.ny && k < g.nz) {
            const long long row = (long long)g.nx * (j + (long long)g.ny * k);
            const int x1 = min(t0x + C::TX, g.nx);
            s0 = (int)cell_offset[row + t0x];
            len = (int)cell_offset[row + x1] - s0;
        }
        seg_start[tid] = s0;
        seg_pref[tid + 1] = len;    // lengths; prefix-summed below
    }
    if (tid == 0) seg_pref[0] = 0;
    __syncthreads();
    if (tid == 0) {
        int run = 0;
        for (int s = 0; s < C::NSEG; ++s) {
            const int len = seg_pref[s + 1];
            seg_pref[s] = run;
            run += len;
        }
        seg_pref[C::NSEG] = run;
    }
    __syncthreads();
    const int n_tile = seg_pref[C::NSEG];
    if (n_tile == 0) return;    // empty tile: nothing to gather, nothing to deposit (block-uniform)
    for (int c = tid; c < C::NCELL; c += C::NT) {
        const int cx = c % C::TX, cy = (c / C::TX) % C::TY, cz = c / (C::TX * C::TY);
        const int i = t0x + cx, j = t0y + cy, k = t0z + cz;
        int lo = 0, hi = 0;
        if (i < g.nx && j < g.ny && k < g.nz) {
            const long long key = i + (long long)g.nx * (j + (long long)g.ny * k);
            const int s = cy + C::TY * cz;
            lo = seg_pref[s] + ((int)cell_offset[key] - seg_start[s]);
            hi = seg_pref[s] + ((int)cell_offset[key + 1] - seg_start[s]);
        }
        cell_lo[c] = lo;
        cell_hi[c] = hi;
    }
    // ---- stage the field stencil, zero the J tile -----------------------------------
    {
        const double* src[6] = {f.Ex, f.Ey, f.Ez, f.Bx, f.By, f.Bz};
        for (int e = tid; e < C::ESZ; e += C::NT) {
            const int ex = e % C::EX, ey = (e / C::EX) % C::EY, ez = e / (C::EX * C::EY);
            const int gx = t0x - C::GL + ex + NG, gy = t0y - C::GL + ey + NG, gz = t0z - C::GL + ez + NG;
            const bool ok = gx >= 0 && gx < g.nx + 2 * NG && gy >= 0 && gy < g.py && gz >= 0 && gz < g.pz;
            const long long o = gx + g.sy * gy + g.sz * gz;
#pragma unroll
            for (int cpt = 0; cpt < 6; ++cpt) Et[cpt * C::ESZ + e] = ok ? __ldg(src[cpt] + o) : 0.0;
        }
        for (int e = tid; e < 3 * C::JSZ; e += C::NT) Jt[e] = 0.0;
    }
    __syncthreads();

    const double inv_c2 = 1.0 / (C_LIGHT * C_LIGHT);
    const double inv_dt = 1.0 / g.dt;
    unsigned int n_fast = 0, n_slow = 0, n_glob = 0;
    bool bad_any = false;

    for (int lo = 0; lo < n_tile; lo += C::CH) {
        const int hi = min(lo + C::CH, n_tile);
        // ---------------- phase A: gather + push + move, particle-major ----------------
        for (int idx = lo + tid; idx < hi; idx += C::NT) {
            int s = 0;
#pragma unroll
            for (int step = C::NSEG / 2; step >= 1; step >>= 1)
                if (s + step < C::NSEG && seg_pref[s + step] <= idx) s += step;
            const long long ip = (long long)seg_start[s] + (idx - seg_pref[s]);
            const int slot = idx - lo, sl = slot + (slot >> 3);
            const double x = p.x[ip], y = p.y[ip], z = p.z[ip];
            const double xi = (x - g.xmin) * g.inv_dx, et = (y - g.ymin) * g.inv_dy, ze = (z - g.zmin) * g.inv_dz;
            const int ci = __double2int_rd(xi), cj = __double2int_rd(et), ck = __double2int_rd(ze);
            const int rx = rel_cell(ci, t0x, C::TX, g.nx), ry = rel_cell(cj, t0y, C::TY, g.ny),
                      rz = rel_cell(ck, t0z, C::TZ, g.nz);
            const bool in_tile = rx >= -DRIFT && rx <= C::TX - 1 + DRIFT && t0x + rx <= g.nx - 1 + DRIFT &&
                                 ry >= -DRIFT && ry <= C::TY - 1 + DRIFT && t0y + ry <= g.ny - 1 + DRIFT &&
                                 rz >= -DRIFT && rz <= C::TZ - 1 + DRIFT && t0z + rz <= g.nz - 1 + DRIFT;
            if (!in_tile) {
                // left the tile's halo since the last sort: whole update against the global arrays
                update_particle_global<N>(g, f, p, ip, q, h, status);
                stg[6 * C::STG + sl] = 0.0;    // nothing to deposit in phase B
                ++n_glob;
                continue;
            }
            double ux = p.ux[ip], uy = p.uy[ip], uz = p.uz[ip];
            const double w = p.w[ip];
            double wxn[N + 1], wyn[N + 1], wzn[N + 1], wxs[N + 1], wys[N + 1], wzs[N + 1];
            // first nodes, shifted from global node index to tile slot: slot = node - (t0 - GL) + (image shift)
            const int shx = (rx - (ci - t0x)) + C::GL - t0x, shy = (ry - (cj - t0y)) + C::GL - t0y,
                      shz = (rz - (ck - t0z)) + C::GL - t0z;
            const int fxn = shape_weights<N>(xi, wxn) + shx, fyn = shape_weights<N>(et, wyn) + shy,
                      fzn = shape_weights<N>(ze, wzn) + shz;
            const int fxs = shape_weights<N>(xi - 0.5, wxs) + shx, fys = shape_weights<N>(et - 0.5, wys) + shy,
                      fzs = shape_weights<N>(ze - 0.5, wzs) + shz;
            const double ex = gather_tile<N, C>(Et + 0 * C::ESZ, fxs, fyn, fzn, wxs, wyn, wzn);
            const double ey = gather_tile<N, C>(Et + 1 * C::ESZ, fxn, fys, fzn, wxn, wys, wzn);
            const double ez = gather_tile<N, C>(Et + 2 * C::ESZ, fxn, fyn, fzs, wxn, wyn, wzs);
            const double bxp = gather_tile<N, C>(Et + 3 * C::ESZ, fxn, fys, fzs, wxn, wys, wzs);
            const double byp = gather_tile<N, C>(Et + 4 * C::ESZ, fxs, fyn, fzs, wxs, wyn, wzs);
            const double bzp = gather_tile<N, C>(Et + 5 * C::ESZ, fxs, fys, fzn, wxs, wys, wzn);
            boris_push(h, inv_c2, ux, uy, uz, ex, ey, ez, bxp, byp, bzp);
            const double gam = sqrt(1.0 + (ux * ux + uy * uy + uz * uz) * inv_c2);
            const double x1 = x + g.dt * ux / gam, y1 = y + g.dt * uy / gam, z1 = z + g.dt * uz / gam;
            const double xi1 = (x1 - g.xmin) * g.inv_dx, et1 = (y1 - g.ymin) * g.inv_dy,
                         ze1 = (z1 - g.zmin) * g.inv_dz;
            const bool bad = !(isfinite(x1) && isfinite(y1) && isfinite(z1)) || !(fabs(xi1 - xi) < 1.0) ||
                             !(fabs(et1 - et) < 1.0) || !(fabs(ze1 - ze) < 1.0);
            bad_any = bad_any || bad;
            p.x[ip] = wrap1(x1, g.xmin, g.xmax, g.Lx);
            p.y[ip] = wrap1(y1, g.ymin, g.ymax, g.Ly);
            p.z[ip] = wrap1(z1, g.zmin, g.zmax, g.Lz);
            p.ux[ip] = ux;
            p.uy[ip] = uy;
            p.uz[ip] = uz;
            stg[0 * C::STG + sl] = xi;
            stg[1 * C::STG + sl] = et;
            stg[2 * C::STG + sl] = ze;
            stg[3 * C::STG + sl] = xi1;
            stg[4 * C::STG + sl] = et1;
            stg[5 * C::STG + sl] = ze1;
            stg[6 * C::STG + sl] = bad ? 0.0 : q * w;
            if (rx == ci - t0x + 0 && ry == cj - t0y && rz == ck - t0z) ++n_fast; else ++n_slow;
        }
        __syncthreads();
        // ---------------- phase B: Esirkepov deposition, cell-major ----------------------
        {
            const int c = tid % C::NCELL, sub = tid / C::NCELL;
            const int p0 = max(cell_lo[c], lo), p1 = min(cell_hi[c], hi);
            for (int idx = p0 + sub; idx < p1; idx += C::NSUB) {
                const int slot = idx - lo, sl = slot + (slot >> 3);
                const double qw = stg[6 * C::STG + sl];
                if (qw == 0.0) continue;
                const double xi = stg[0 * C::STG + sl], et = stg[1 * C::STG + sl], ze = stg[2 * C::STG + sl];
                const double xi1 = stg[3 * C::STG + sl], et1 = stg[4 * C::STG + sl], ze1 = stg[5 * C::STG + sl];
                double s0x[N + 2], dsx[N + 2], s0y[N + 2], dsy[N + 2], s0z[N + 2], dsz[N + 2];
                bool bad = false;
                const int nx0 = shapes_pair<N>(xi, xi1, s0x, dsx, bad);
                const int ny0 = shapes_pair<N>(et, et1, s0y, dsy, bad);
                const int nz0 = shapes_pair<N>(ze, ze1, s0z, dsz, bad);
                // image shift of the OLD cell, as in phase A
                const int ci = __double2int_rd(xi), cj = __double2int_rd(et), ck = __double2int_rd(ze);
                const int ox = nx0 + (rel_cell(ci, t0x, C::TX, g.nx) - ci) + C::JL;
                const int oy = ny0 + (rel_cell(cj, t0y, C::TY, g.ny) - cj) + C::JL;
                const int oz = nz0 + (rel_cell(ck, t0z, C::TZ, g.nz) - ck) + C::JL;
                const double cqx = -qw * inv_dt * g.inv_dy * g.inv_dz;
                const double cqy = -qw * inv_dt * g.inv_dx * g.inv_dz;
                const double cqz = -qw * inv_dt * g.inv_dx * g.inv_dy;
                deposit_tile<N, C>(Jt, ox, oy, oz, s0x, dsx, s0y, dsy, s0z, dsz, cqx, cqy, cqz);
            }
        }
        __syncthreads();
    }
    // ---- flush: one global atomic per non-zero tile point ---------------------------------
    {
        double* dst[3] = {f.Jx, f.Jy, f.Jz};
        for (int e = tid; e < C::JSZ; e += C::NT) {
            const int jx = e % C::JX, jy = (e / C::JX) % C::JY, jz = e / (C::JX * C::JY);
            const int gx = t0x - C::JL + jx + NG, gy = t0y - C::JL + jy + NG, gz = t0z - C::JL + jz + NG;
            const bool ok = gx >= 0 && gx < g.nx + 2 * NG && gy >= 0 && gy < g.py && gz >= 0 && gz < g.pz;
            if (!ok) continue;
            const long long o = gx + g.sy * gy + g.sz * gz;
#pragma unroll
            for (int cpt = 0; cpt < 3; ++cpt) {
                const double v = Jt[cpt * C::JSZ + e];
                if (v != 0.0) atomicAdd(dst[cpt] + o, v);
            }
        }
    }
    // ---- counters ----------------------------------------------------------------------------
    if (bad_any) status->ephys = 1;
    n_fast = __reduce_add_sync(0xffffffffu, n_fast);
    n_slow = __reduce_add_sync(0xffffffffu, n_slow);
    n_glob = __reduce_add_sync(0xffffffffu, n_glob);
    if ((tid & 31) == 0) {
        if (n_fast) atomicAdd(&status->n_fast, (unsigned long long)n_fast);
        if (n_slow) atomicAdd(&status->n_slow, (unsigned long long)n_slow);
        if (n_glob) atomicAdd(&status->n_global, (unsigned long long)n_glob);
    }
}

using Cfg = TileCfg<8, 4, 4, 256, 512>;

template <int N>
void launch_tile(const Grid& g, const Fields& f, const Particles& p, double q, double h,
                 const unsigned int* cell_offset, DevStatus* status, cudaStream_t st) {
    const int ntx = (g.nx + Cfg::TX - 1) / Cfg::TX, nty = (g.ny + Cfg::TY - 1) / Cfg::TY,
              ntz = (g.nz + Cfg::TZ - 1) / Cfg::TZ;
    const long long nb = (long long)ntx * nty * ntz;
    particles_tile_kernel<N, Cfg><<<(unsigned)nb, Cfg::NT, Cfg::SMEM, st>>>(g, f, p, q, h, cell_offset, ntx, nty,
                                                                           status);
}

}  // namespace

int tile_setup() {
    cudaError_t e = cudaFuncSetAttribute(particles_tile_kernel<1, Cfg>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)Cfg::SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(particles_tile_kernel<2, Cfg>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)Cfg::SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(particles_tile_kernel<3, Cfg>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)Cfg::SMEM);
    return (int)e;
}

int launch_particles_tile(const Grid& g, const Fields& f, const Particles& p, long long n, double q, double m,
                          int order, const unsigned int* cell_offset, DevStatus* status, cudaStream_t st) {
    if (n <= 0) return 0;
    const double h = q * g.dt / (2.0 * m);
    if (order == 1) launch_tile<1>(g, f, p, q, h, cell_offset, status, st);
    else if (order == 2) launch_tile<2>(g, f, p, q, h, cell_offset, status, st);
    else launch_tile<3>(g, f, p, q, h, cell_offset, status, st);
    return 1;
}

}  // namespace pic
