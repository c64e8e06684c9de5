// particles_tile.cu -- fused gather + Boris push + Esirkepov deposition per
// cell-sorted tile (BASELINE.json:north_star parts
// 1-3, "fused per cell-sorted tile").  Kernel v9 of DESIGN.md section 5.1;
// measurements in profiles/r02_tile_kernel.md (v1-v8: profiles/r01_summary.md).
//
// One thread block owns a tile of TX x TY x TZ cells; its E,B stencil (+ halo
// for the shape support and DRIFT cells of drift since the last pic_sort) is
// staged in shared memory once.  After that the block's warps run without any
// block-wide barrier, as NP producer / consumer PAIRS: a producer warp runs
// phase A, its consumer warp phase B and the flush, concurrently, on a per-pair
// staging ring in shared memory handed over with st.release / ld.acquire
// counters (positions staged, positions consumed).  Neither role keeps the
// other's registers alive: 168 registers and 12 warps per SM instead of 255 and 8.
// A producer owns RPW consecutive x-rows of the tile; their cells, in order,
// form its STREAM: cell c occupies the stream positions cp[c] .. cp[c] + n_c - 1.
//   phase A  (producer) lane <-> stream position, 32 consecutive positions at a time,
//            ACROSS row boundaries (the lanes stay full: a row of 64 +- 8
//            particles no longer ends in a nearly empty sub-chunk).  The
//            particle data of a sub-chunk are copied into a per-warp landing
//            buffer by cp.async one sub-chunk ahead (with a deferred sort
//            pending: through perm[], read two sub-chunks ahead, and all eight
//            arrays are then written, in sorted order, to the other buffer).
//            Gather from the shared stencil, Boris, move, store of the wrapped
//            state.  A particle that stayed inside its listed cell or crossed
//            ONE of its faces ("fast") writes its old nodal shapes and shape
//            differences on the cell's window to slot (position mod RING) of a
//            per-warp staging ring: 18 doubles (the last entry of each set
//            follows from sum S = 1, sum DS = 0) + (q w / dt, e) + a code.
//   phase B  (consumer) runs as soon as a whole row is staged (or the ring is full):
//            lane <-> (cell q of the row, plane s of that cell's window).  The
//            four lanes of a cell walk the cell's staged particles and
//            accumulate the Esirkepov window of the CELL in registers
//            (3 x 12 accumulators per lane at order 3), so the per-particle
//            cost is FMAs and shared-memory loads, not atomics.
//   slow     a particle that crossed several faces or is not in its listed
//            cell stages its positions and is deposited by the whole producer warp: its
//            (N+2)^3 window is spread over the lanes, one global RED.ADD.F64
//            per non-zero point.
//   flush    at the end of a row the lanes add up, with shuffles, what lands on
//            the same global node and issue one RED.ADD.F64 per distinct node
//            (fire-and-forget; fp64 atomicAdd on SHARED memory is a CAS loop on
//            sm_100a, which is why there is no shared J tile).
// A particle outside the tile's halo gathers from global memory instead; the
// kernel is correct for any particle order, only slower (R39).
#include "particle_update.cuh"

namespace pic {

namespace {

template <int N>
struct FastWin {
    static constexpr int FW = (N == 1) ? 2 : 4;    // nodes of the per-cell window (old and new cell identical)
    static constexpr int FA = (N == 1) ? 0 : -1;   // first window node relative to the cell index
};

// DRIFT = cells a particle may sit outside the tile and still gather from shared memory: 1 for a species
// that has moved since its last pic_sort, 0 right after a sort (every particle is in its listed cell), which
// shrinks the stencil from 14 x 10 x 10 to 12 x 8 x 8 nodes per component so that TWO blocks fit one SM
// and one block's prologue (stencil staging: every warp of the block waits) overlaps the other's particles.
template <int TX_, int TY_, int TZ_, int NP_, int MINB_, int DRIFT_, int RING_, class FT_ = double>
struct TileCfg {
    // FT = type of the staged field stencil and of the gather / push arithmetic: double, or float in the
    // mixed-precision mode (pic_set_option "precision" = 1)
    using FT = FT_;
    // NP producer warps (phase A) and NP consumer warps (phase B), paired one to one
    static constexpr int TX = TX_, TY = TY_, TZ = TZ_, NP = NP_, NW = 2 * NP_, NT = 32 * NW, MINB = MINB_,
                         DRIFT = DRIFT_;
    // The consumer starts on an unfinished row once its producer is within AHEAD records of running out of ring space:
    // 32 (one sub-chunk, i.e. when the producer is about to block) leaves the producers waiting 6 % of their time, 64
    // halves that for a few more partial passes (31.0 instead of 31.9 ms per step; 80: 31.6, 96: 32.1).
    static constexpr int AHEAD = 64;
    static constexpr unsigned POLL_NS = 800;      // consumer's poll interval while its producer is still staging the row
    static constexpr int NROW = TY * TZ;
    // gather stencil: nodes i-2 .. i+2 of a particle in cell i (every order, every staggering)
    static constexpr int GL = 2 + DRIFT;
    static constexpr int EX = TX + 2 * GL, EY = TY + 2 * GL, EZ = TZ + 2 * GL;
    static constexpr int ESZ = EX * EY * EZ;      // nodes per component
    // Shared layout: word(x, y, z) = y + SZ z + SX x (y fastest, x slowest).  The addresses one gather load
    // touches in a half-warp -- a few adjacent cells in x, times the -1/0 stagger shift in every dimension --
    // must fall into 16 different 8-byte banks: (SZ, SX) = (10, 4) or (8, 2) mod 16 does that.
    static constexpr int SZ = EY;
    static constexpr int SXR = (SZ % 16 == 10) ? 4 : 2;
    static constexpr int SX = EZ * SZ + ((SXR - (EZ * SZ) % 16) + 16) % 16;
    static_assert(SZ % 16 == 10 || SZ % 16 == 8, "no conflict-free stride for this tile height");
    // One component occupies FP words; components that are nodal in x (Ey, Ez, Bx) never read x-slab 0
    // (their lowest node is i-1), so that slab is not stored: their base is shifted back by one slab.
    static constexpr int FP = (EX - 1) * SX + (EZ - 1) * SZ + EY;
    static constexpr int TOT = 6 * FP - 3 * SX + ((6 * FP - 3 * SX) & 1);     // stencil words of type FT, even
    // the stencil in units of doubles, rounded up to a 16-byte boundary: staging stays 16-byte aligned
    static constexpr int TOT_D = ((TOT * (int)sizeof(FT) + 15) / 16) * 2;
    __host__ __device__ static constexpr bool trimmed(int k) { return k >= 1 && k <= 3; }
    __host__ __device__ static constexpr int comp_base(int k) {   // word of (x = 0, y = 0, z = 0), virtual for k = 1..3
        return k == 0 ? 0 : (k == 1 ? FP - SX : (k == 2 ? 2 * FP - 2 * SX : (k == 3 ? 3 * FP - 3 * SX
                      : (k == 4 ? 4 * FP - 3 * SX : 5 * FP - 3 * SX))));
    }
    // a producer's stream: RPW rows of the tile, NC cells
    static constexpr int RPW = NROW / NP, NC = RPW * TX;
    static_assert(NROW % NP == 0 && NC <= 64, "rows are dealt statically; one lane scans two cells of the stream");
    // per-pair staging ring of RING slots: a body of BODY doubles per slot (slot s at word BODY s + 2 (s >> 3): BODY / 2
    // is odd and every eighth slot is pushed on by one 16-byte word, so that the eight 16-byte words a phase-B warp
    // load touches -- slots about 8 apart -- fall into different 16-byte bank groups), a tail (q w / dt, e) and a
    // code per slot; then the scratch record of the slow path, the landing buffer of the next sub-chunk's particle
    // data (8 arrays x 32 lanes, filled by cp.async), the stream table cp[NC + 1] and the pair's two flags.
    static constexpr int RING = RING_, BODY = 18, SLOW_W = 32, PBUF_W = 8 * 32;
    static constexpr int BODY_W = BODY * RING + 2 * ((RING + 7) / 8), TAIL_W = 2 * RING, CODE_W = (RING + 1) / 2,
                         TAB_W = (NC + 1 + 4 + 4) / 2 + ((NC + 1 + 4 + 4) / 2 & 1);
    static constexpr int STG_W = BODY_W + TAIL_W + CODE_W + (CODE_W & 1) + SLOW_W + PBUF_W + TAB_W;
    static_assert(STG_W % 2 == 0 && BODY_W % 2 == 0, "staging layout: 16-byte alignment");
    static constexpr int NOFF = NROW * (TX + 1);
    static constexpr size_t SMEM = sizeof(double) * ((size_t)TOT_D + (size_t)NP * STG_W) + sizeof(int) * (NOFF + 4);
    static_assert(TX == 8, "phase B maps 8 cells x 4 planes onto a warp");
};

// word offset of ring slot s inside the body area
template <class C>
__device__ __forceinline__ int body_word(int s) { return C::BODY * s + 2 * (s >> 3); }


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

// N+1 weights whose first node is `first`, placed on the per-cell window that starts at node `anchor`.
template <int N>
__device__ __forceinline__ void to_fast_window(const double (&w)[N + 1], int first, int anchor,
                                               double (&out)[FastWin<N>::FW]) {
    if constexpr (N == 2) {
        const bool up = first != anchor;    // base = floor(xi + 1/2) is the cell's upper node
        out[0] = up ? 0.0 : w[0];
        out[1] = up ? w[0] : w[1];
        out[2] = up ? w[1] : w[2];
        out[3] = up ? w[2] : 0.0;
    } else {
#pragma unroll
        for (int a = 0; a <= N; ++a) out[a] = w[a];
    }
}

// N+1 new weights whose first node sits sh = first - anchor slots into the per-cell window (sh = -1 .. 2
// for a move of less than one cell): weights landing on slots 0 .. FW-1 go to out[], the one that may land
// on slot -1 or FW (the particle crossed the cell face) is returned in e_lo / e_hi.
template <int N>
__device__ __forceinline__ void place_new_window(const double (&w)[N + 1], int sh, double (&out)[FastWin<N>::FW],
                                                 double& e_lo, double& e_hi) {
    constexpr int FW = FastWin<N>::FW;
    constexpr int TMAX = (N == 2) ? 2 : 1;    // orders 1 and 3 anchor their support at floor(xi): sh = -1, 0 or 1
#pragma unroll
    for (int a = 0; a < FW; ++a) {
        double v = 0.0;
#pragma unroll
        for (int t = -1; t <= TMAX; ++t) {
            const int k = a - t;                      // weight index that lands on slot a when sh == t
            if (k >= 0 && k <= N) v = (sh == t) ? w[k] : v;
        }
        out[a] = v;
    }
    e_lo = (sh == -1) ? w[0] : 0.0;
    e_hi = 0.0;
#pragma unroll
    for (int t = 0; t <= TMAX; ++t) {
        const int k = FW - t;
        if (k >= 0 && k <= N) e_hi = (sh == t) ? w[k] : e_hi;
    }
}

// Shared stencil layout (TileCfg): word(x, y, z) = y + SZ z + SX x, conflict-free strides (the x-fastest
// layout had 1.4x-1.7x wavefronts on the components staggered in y).
template <class C>
__device__ __forceinline__ int tile_word(int x, int y, int z) { return y + C::SZ * z + C::SX * x; }

// One z-plane of one component from the shared stencil: sum_b wy[b] sum_a wx[a] F[a,b].
template <int WX, int WY, int PX, int PY, class C, class T>
__device__ __forceinline__ T gather_plane(const T* __restrict__ base, const T (&wx)[PX], const T (&wy)[PY]) {
    T accy = T(0);
#pragma unroll
    for (int b = 0; b < WY; ++b) {
        T accx = T(0);
#pragma unroll
        for (int a = 0; a < WX; ++a) accx = fma_t(wx[a], base[b + C::SX * a], accx);
        accy = fma_t(wy[b], accx, accy);
    }
    return accy;
}

// All six components on the particle's own windows (N + 1 nodes, NS + 1 along staggered directions): 384 loads at
// order 3, at 1.8 wavefronts each.  (Cell-anchored windows, 540 loads at one wavefront each, were measured slower
// in round 2 and removed in round 3: DESIGN.md 5.1, profiles/r02_lsu.md.)  (g*n) / (f*s) = tile slot of the first nodal / staggered node per
// dimension.  The z weights rotate through arrays padded to ZT = N + 1 entries.
template <int N, int GV, class C>
__device__ __forceinline__ void gather6_part(const typename C::FT* __restrict__ Et, int gxn, int gyn, int gzn, int fxs,
                                             int fys, int fzs, const typename C::FT (&wxn)[N + 1],
                                             const typename C::FT (&wyn)[N + 1], typename C::FT (&wzn)[N + 1],
                                             const typename C::FT (&wxs)[GatherOrders<N, GV>::NS + 1],
                                             const typename C::FT (&wys)[GatherOrders<N, GV>::NS + 1],
                                             typename C::FT (&wzs)[N + 1], typename C::FT (&eb)[6]) {
    using FT = typename C::FT;
    constexpr int WN = N + 1, WS = GatherOrders<N, GV>::NS + 1;
    const int o_ex = C::comp_base(0) + tile_word<C>(fxs, gyn, gzn);
    const int o_ey = C::comp_base(1) + tile_word<C>(gxn, fys, gzn);
    const int o_ez = C::comp_base(2) + tile_word<C>(gxn, gyn, fzs);
    const int o_bx = C::comp_base(3) + tile_word<C>(gxn, fys, fzs);
    const int o_by = C::comp_base(4) + tile_word<C>(fxs, gyn, fzs);
    const int o_bz = C::comp_base(5) + tile_word<C>(fxs, fys, gzn);
#pragma unroll
    for (int k = 0; k < 6; ++k) eb[k] = FT(0);
    const FT* pl = Et;
#pragma unroll 1
    for (int c = 0; c < WN; ++c, pl += C::SZ) {
        const FT zn = wzn[0], zs = wzs[0];
        eb[0] = fma_t(zn, gather_plane<WS, WN, WS, WN, C, FT>(pl + o_ex, wxs, wyn), eb[0]);
        eb[1] = fma_t(zn, gather_plane<WN, WS, WN, WS, C, FT>(pl + o_ey, wxn, wys), eb[1]);
        eb[5] = fma_t(zn, gather_plane<WS, WS, WS, WS, C, FT>(pl + o_bz, wxs, wys), eb[5]);
        if (WS == WN || c < WS) {
            eb[2] = fma_t(zs, gather_plane<WN, WN, WN, WN, C, FT>(pl + o_ez, wxn, wyn), eb[2]);
            eb[3] = fma_t(zs, gather_plane<WN, WS, WN, WS, C, FT>(pl + o_bx, wxn, wys), eb[3]);
            eb[4] = fma_t(zs, gather_plane<WS, WN, WS, WN, C, FT>(pl + o_by, wxs, wyn), eb[4]);
        }
#pragma unroll
        for (int k = 0; k < N; ++k) { wzn[k] = wzn[k + 1]; wzs[k] = wzs[k + 1]; }
        wzn[N] = zn;
        wzs[N] = zs;
    }
}

// Gather of all six components from the padded GLOBAL arrays (particle outside the tile's halo).
template <int N, int GV, class T>
__device__ __noinline__ void gather_global6(const Grid& g, const Fields& f, double xi, double et, double ze,
                                            T (&eb)[6]) {
    gather6_global<N, GV, T>(g, f, xi, et, ze, eb);
}

// tile-relative cell index with the periodic image nearest to the tile
template <int DRIFT>
__device__ __forceinline__ int rel_cell(int i, int t0, int T, int n) {
    int r = i - t0;
    if (r < -DRIFT) r += n;
    else if (r > T - 1 + DRIFT) r -= n;
    return r;
}

}  // namespace

namespace {

constexpr int REC_FAST = 0;   // fast record (FastRec layout): old and new cell identical
// 1 .. 6: fast record of a particle that crossed ONE cell face: 1 + 2 d + (1 if towards +d).  The part of
// its Esirkepov window inside the cell's window is in the record; the one node layer outside it carries
// S0 = 0, DS = e (the new weight that left the window; tail.y of the slot).
constexpr int REC_NONE = 7;   // nothing to deposit (q = 0, or the particle raised PIC_EPHYS)
constexpr int REC_SLOW = 8;   // slow particle: the slot holds xi0 eta0 zeta0 xi1 eta1 zeta1 qw; deposited by the whole warp

// fp64 add to GLOBAL memory without a return value: REDG.E.ADD.F64 (fire-and-forget).  atomicAdd on a
// pointer whose address space the compiler cannot prove emits a generic ATOM with a returned value
// plus shared-memory CAS fallbacks, and every use then waits a full L2 round trip.
__device__ __forceinline__ void red_add(double* p, double v) {
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory");
}


// pull one 32-particle sub-chunk of the SoA arrays towards the SM ahead of its use
// A load the compiler must issue HERE (it otherwise sinks the load next to its first use, which is the point
// where the latency was meant to be over).
__device__ __forceinline__ int ld_u32_now(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.global.nc.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return (int)v;
}

// 8-byte asynchronous copy global -> shared (LDGSTS): the data land in shared memory without a register
// and without a scoreboard wait in the issuing warp
__device__ __forceinline__ void cp_async8(double* dst_smem, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(dst_smem)), "l"(src)
                 : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

__device__ __forceinline__ double2 ld2(const double* r, int i) { return *reinterpret_cast<const double2*>(r + i); }
__device__ __forceinline__ void st2(double* r, int i, double a, double b) {
    *reinterpret_cast<double2*>(r + i) = make_double2(a, b);
}

// ---- slow path: one particle deposited by the whole warp -----------------------------------
template <int N>
struct SlowRec {
    static constexpr int W = N + 2;
    // per dimension d: s0 at 2 W d, ds at 2 W d + W;  then -q w / dt and the window's first padded offset
    static constexpr int S0X = 0, DSX = W, S0Y = 2 * W, DSY = 3 * W, S0Z = 4 * W, DSZ = 5 * W, CQ = 6 * W,
                         ORG = 6 * W + 1;
    static_assert(ORG < 32, "slow record larger than the scratch area");
};

// The staging slot of a slow particle holds only (xi0, eta0, zeta0, xi1, eta1, zeta1, q w).  Lanes 0..2 expand
// it, one dimension each, into the SlowRec of the warp's scratch area.  Called by all 32 lanes.
template <int N>
__device__ __forceinline__ void slow_build(const double* slot, double* rec, const Grid& g, double inv_dt, int lane) {
    using R = SlowRec<N>;
    constexpr int W = R::W;
    long long o = 0;
    if (lane < 3) {
        const int d = lane;
        const long long stride = (d == 0) ? 1 : ((d == 1) ? g.sy : g.sz);
        double s0[W], ds[W];
        bool bad = false;
        const int n0 = shapes_pair<N>(slot[d], slot[3 + d], s0, ds, bad);
        double* r = rec + 2 * W * d;
#pragma unroll
        for (int a = 0; a < W; ++a) { r[a] = s0[a]; r[W + a] = ds[a]; }
        o = stride * (long long)(n0 + NG);     // window nodes stay inside the guard shell
    }
    const long long o1 = __shfl_down_sync(0xffffffffu, o, 1), o2 = __shfl_down_sync(0xffffffffu, o, 2);
    if (lane == 0) {
        rec[R::CQ] = -slot[6] * inv_dt;
        rec[R::ORG] = __longlong_as_double(o + o1 + o2);
    }
    __syncwarp();
}

// Called by all 32 lanes: lane <-> one (u,v) pair of the window's cross-section; W-1 points along the
// prefix direction each.  Jx = cqx prefix_a(DSx) (S0y Az + DSy Bz), A = S0 + DS/2, B = S0/2 + DS/3, and
// cyclic permutations.  Rolled over the three components.
template <int N>
__device__ __forceinline__ void slow_deposit(const double* rec, const Grid& g, const Fields& f, int lane) {
    using R = SlowRec<N>;
    constexpr int W = R::W;
    if (lane >= W * W) return;
    const int u = lane % W, v = lane / W;
    const long long o0 = __double_as_longlong(rec[R::ORG]);
    const double cq0 = rec[R::CQ];
    const double third = 1.0 / 3.0;
#pragma unroll 1
    for (int d = 0; d < 3; ++d) {
        // component d: prefix along d; (u,v) run over the other two dimensions (e1 < e2)
        const int e1 = (d == 0) ? 1 : 0, e2 = (d == 2) ? 1 : 2;
        const long long sd = (d == 0) ? 1 : ((d == 1) ? g.sy : g.sz);
        const long long s1 = (e1 == 0) ? 1 : g.sy, s2 = (e2 == 1) ? g.sy : g.sz;
        const double a2 = rec[2 * W * e2 + v], b2 = rec[2 * W * e2 + W + v];
        const double t = rec[2 * W * e1 + u] * (a2 + 0.5 * b2) + rec[2 * W * e1 + W + u] * (0.5 * a2 + third * b2);
        if (t != 0.0) {
            const double cq = cq0 * ((d == 0) ? g.inv_dy * g.inv_dz : ((d == 1) ? g.inv_dx * g.inv_dz
                                                                                 : g.inv_dx * g.inv_dy));
            double* dst = ((d == 0) ? f.Jx : ((d == 1) ? f.Jy : f.Jz)) + o0 + s1 * u + s2 * v;
            const double* dsd = rec + 2 * W * d + W;
            double acc = 0.0;
#pragma unroll
            for (int a = 0; a < W - 1; ++a) {
                acc += dsd[a];
                const double val = (cq * acc) * t;
                if (val != 0.0) red_add(dst + sd * a, val);
            }
        }
    }
}

// ---- fast path: per-(cell, plane) register accumulators --------------------------------------
// Staging slot body (FW = window nodes): for d = x, y, z the first FW - 1 entries of S0_d, then of DS_d; the last
// entry of each set follows from sum_a S0[a] = 1 and sum_a DS[a] = -e_d (e_d = the new weight of a face crosser
// that left the window in dimension d, else 0).  The tail holds -q w / dt and e.  The prefix-summed current factors
// pd_d[a] = cq_d * sum_{a' <= a} ds_d[a'] are rebuilt by the phase-B lanes (18 fp64 operations) instead of
// being staged (9 more doubles per particle through the shared-memory pipe, which is what binds the kernel).
template <int N>
struct FastRec {
    static constexpr int FW = FastWin<N>::FW, M = FW - 1;
    static constexpr int LEN = 6 * M;
    __host__ __device__ static constexpr int s0(int d, int a) { return 2 * M * d + a; }
    __host__ __device__ static constexpr int ds(int d, int a) { return 2 * M * d + M + a; }
};

template <int K>
__device__ __forceinline__ double pick(const double (&v)[K], int s) {
    double r = v[0];
#pragma unroll
    for (int k = 1; k < K; ++k) r = (s == k) ? v[k] : r;
    return r;
}

template <int N>
struct CellAcc {
    static constexpr int FW = FastWin<N>::FW;
    static constexpr int NACC = 3 * FW * (FW - 1);
    double jx[FW][FW - 1];   // Jx[b][a] on plane c = s
    double jy[FW - 1][FW];   // Jy[b][a] on plane c = s
    double jz[FW - 1][FW];   // Jz[c][a] on row   b = s
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int b = 0; b < FW; ++b)
#pragma unroll
            for (int a = 0; a < FW - 1; ++a) { jx[b][a] = 0.0; jy[a][b] = 0.0; jz[a][b] = 0.0; }
    }
    // one staged particle; s = this lane's plane.  Returns false for a record that is not fast.
    // r = the slot's body, tail = (-q w / dt, e), code = the slot's code; jx0, jy0, jz0 = global J pointers at
    // the first node of this cell's window (for the crosser's overflow layer).
    __device__ __forceinline__ bool add(const double* __restrict__ r, double2 tail, int code, int s,
                                        double* jx0, double* jy0, double* jz0, long long sy, long long sz,
                                        double area_x, double area_y, double area_z) {
        using R = FastRec<N>;
        const double third = 1.0 / 3.0;
        if (code >= REC_NONE) return false;
        double raw[R::LEN];
#pragma unroll
        for (int k = 0; k < R::LEN; k += 2) {
            const double2 v = ld2(r, k);
            raw[k] = v.x; raw[k + 1] = v.y;
        }
        // a face crosser's prefix starts with the weight that fell below the window in the crossed dimension
        const double e = tail.y;
        const double ex = (code == 1 || code == 2) ? e : 0.0, ey = (code == 3 || code == 4) ? e : 0.0,
                     ez = (code == 5 || code == 6) ? e : 0.0;
        const double e0x = (code == 1) ? e : 0.0, e0y = (code == 3) ? e : 0.0, e0z = (code == 5) ? e : 0.0;
        double s0x[FW], dsx[FW], s0y[FW], dsy[FW], s0zz[FW], dsz[FW], pdx[FW - 1], pdy[FW - 1], pdz[FW - 1];
        {
            double tx0 = 1.0, tx1 = -ex, ty0 = 1.0, ty1 = -ey, tz0 = 1.0, tz1 = -ez;
#pragma unroll
            for (int a = 0; a < FW - 1; ++a) {
                s0x[a] = raw[R::s0(0, a)]; dsx[a] = raw[R::ds(0, a)];
                s0y[a] = raw[R::s0(1, a)]; dsy[a] = raw[R::ds(1, a)];
                s0zz[a] = raw[R::s0(2, a)]; dsz[a] = raw[R::ds(2, a)];
                tx0 -= s0x[a]; tx1 -= dsx[a]; ty0 -= s0y[a]; ty1 -= dsy[a]; tz0 -= s0zz[a]; tz1 -= dsz[a];
            }
            s0x[FW - 1] = tx0; dsx[FW - 1] = tx1; s0y[FW - 1] = ty0; dsy[FW - 1] = ty1;
            s0zz[FW - 1] = tz0; dsz[FW - 1] = tz1;
        }
        const double s0z = pick<FW>(s0zz, s);
        // outer prefix factor of a face crosser: the prefix over every node below the outer layer is e (towards -d:
        // the layer comes first) or -e (towards +d: all DS sum to zero and the layer's own DS is e)
        const double pd_ov = ((code & 1) ? e : -e) * tail.x *
                             ((code <= 2) ? area_x : ((code <= 4) ? area_y : area_z));
        {
            const double cqx = tail.x * area_x, cqy = tail.x * area_y, cqz = tail.x * area_z;
            double rx = e0x, ry = e0y, rz = e0z;
#pragma unroll
            for (int a = 0; a < FW - 1; ++a) {
                rx += dsx[a]; ry += dsy[a]; rz += dsz[a];
                pdx[a] = cqx * rx; pdy[a] = cqy * ry; pdz[a] = cqz * rz;
            }
        }
        const double dsz_s = pick<FW>(dsz, s);
        const double az = s0z + 0.5 * dsz_s, bz = 0.5 * s0z + third * dsz_s;
        const double s0ys = pick<FW>(s0y, s), dsys = pick<FW>(dsy, s);
        const double ay = s0ys + 0.5 * dsys, by = 0.5 * s0ys + third * dsys;
        double tx[FW], ty[FW], tz[FW];   // cross-section factors of Jx (per b), Jy (per a), Jz (per a)
#pragma unroll
        for (int b = 0; b < FW; ++b) {
            tx[b] = s0y[b] * az + dsy[b] * bz;
#pragma unroll
            for (int a = 0; a < FW - 1; ++a) jx[b][a] = fma(pdx[a], tx[b], jx[b][a]);
        }
#pragma unroll
        for (int a = 0; a < FW; ++a) {
            ty[a] = s0x[a] * az + dsx[a] * bz;
#pragma unroll
            for (int b = 0; b < FW - 1; ++b) jy[b][a] = fma(pdy[b], ty[a], jy[b][a]);
        }
#pragma unroll
        for (int a = 0; a < FW; ++a) {
            tz[a] = s0x[a] * ay + dsx[a] * by;
#pragma unroll
            for (int c = 0; c < FW - 1; ++c) jz[c][a] = fma(pdz[c], tz[a], jz[c][a]);
        }
        if (code != REC_FAST) {
            // ---- face crosser: the node layer just outside the window (S0 = 0, DS = e) ----------------
            const int k = code - 1, d = k >> 1, hi = k & 1;
            const long long node = hi ? FW : -1;          // node slot of the layer
            const long long edge = hi ? FW - 1 : -1;      // edge slot between the layer and the window
            const double he = 0.5 * e, te = third * e;
            if (d == 0) {
                double* px = jx0 + edge + sz * s;
#pragma unroll
                for (int b = 0; b < FW; ++b) red_add(px + sy * b, pd_ov * tx[b]);
                double* py = jy0 + node + sz * s;
                const double ebz = e * bz;
#pragma unroll
                for (int b = 0; b < FW - 1; ++b) red_add(py + sy * b, pdy[b] * ebz);
                double* pz = jz0 + node + sy * s;
                const double eby = e * by;
#pragma unroll
                for (int c = 0; c < FW - 1; ++c) red_add(pz + sz * c, pdz[c] * eby);
            } else if (d == 1) {
                double* py = jy0 + sy * edge + sz * s;
#pragma unroll
                for (int a = 0; a < FW; ++a) red_add(py + a, pd_ov * ty[a]);
                double* px = jx0 + sy * node + sz * s;
                const double ebz = e * bz;
#pragma unroll
                for (int a = 0; a < FW - 1; ++a) red_add(px + a, pdx[a] * ebz);
                if (s < FW - 1) {     // the layer's Jz row belongs to no lane: lane s takes plane c = s
                    double* pz = jz0 + sy * node + sz * s;
                    const double pc = pick<FW - 1>(pdz, s);
#pragma unroll
                    for (int a = 0; a < FW; ++a) red_add(pz + a, pc * (s0x[a] * he + dsx[a] * te));
                }
            } else {
                double* pz = jz0 + sy * s + sz * edge;
#pragma unroll
                for (int a = 0; a < FW; ++a) red_add(pz + a, pd_ov * tz[a]);
                double* px = jx0 + sy * s + sz * node;      // the layer's Jx, Jy planes: lane s takes row b = s
                const double t = s0ys * he + dsys * te;
#pragma unroll
                for (int a = 0; a < FW - 1; ++a) red_add(px + a, pdx[a] * t);
                if (s < FW - 1) {
                    double* py = jy0 + sy * s + sz * node;
                    const double pb = pick<FW - 1>(pdy, s);
#pragma unroll
                    for (int a = 0; a < FW; ++a) red_add(py + a, pb * (s0x[a] * he + dsx[a] * te));
                }
            }
        }
        return true;
    }
    // One x-line of window values v[a] (node or edge q + FA + a of the cell q = lane >> 2) from all eight cells
    // of the row: the windows of neighbouring cells overlap in all but one node, so the lanes first add up,
    // with shuffles, everything that lands on the same global node -- lane q ends up with the total for
    // node q (a = A0 = -FA of its own window) -- and then issue ONE RED per distinct node (10 or 11 per line
    // instead of 24 or 32).  p0 = address of this lane's node q on the line.  Called by all 32 lanes.
    template <int NA, int A0>
    static __device__ __forceinline__ void flush_line(const double (&v)[NA], double* p0, int lane, bool active) {
        const int q = lane >> 2;
        double m = v[A0];
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            if (a == A0) continue;
            const int dq = A0 - a;                      // v[a] of cell q + dq lands on node q
            const double t = __shfl_sync(0xffffffffu, v[a], (lane + 4 * dq) & 31);
            if (q + dq >= 0 && q + dq <= 7) m += t;
        }
        if (active && m != 0.0) red_add(p0, m);
        // nodes outside 0 .. 7: -1 (cell 0, a = 0) and 8 (cell 7, a = A0 + 1; cell 6, a = A0 + 2) in one
        // RED instruction, 9 (cell 7, a = A0 + 2) in another
        double e = 0.0;
        if constexpr (A0 + 2 < NA) e = __shfl_sync(0xffffffffu, v[A0 + 2], (lane - 4) & 31);
        if constexpr (A0 + 1 < NA) e += v[A0 + 1];
        if constexpr (A0 >= 1) e = (q == 0) ? v[0] : e;
        if (active && (q == 7 || (A0 >= 1 && q == 0)) && e != 0.0) red_add(q == 0 ? p0 - 1 : p0 + 1, e);
        if constexpr (A0 + 2 < NA)
            if (active && q == 7 && v[A0 + 2] != 0.0) red_add(p0 + 2, v[A0 + 2]);
    }
    // Add the row's accumulators to the padded global arrays.  o = offset of this lane's window's first node,
    // s = this lane's plane.  Called by all 32 lanes (lanes with s >= FW hold zeros and only shuffle).
    __device__ __forceinline__ void flush(const Grid& g, const Fields& f, long long o, int s, int lane) const {
        constexpr int A0 = -FastWin<N>::FA;
        const bool active = s < FW;
        double* px = f.Jx + o + g.sz * s + A0;
#pragma unroll
        for (int b = 0; b < FW; ++b) flush_line<FW - 1, A0>(jx[b], px + g.sy * b, lane, active);
        double* py = f.Jy + o + g.sz * s + A0;
#pragma unroll
        for (int b = 0; b < FW - 1; ++b) flush_line<FW, A0>(jy[b], py + g.sy * b, lane, active);
        double* pz = f.Jz + o + g.sy * s + A0;
#pragma unroll
        for (int c = 0; c < FW - 1; ++c) flush_line<FW, A0>(jz[c], pz + g.sz * c, lane, active);
    }
};

}  // namespace

namespace {

// ---- flags of a producer / consumer pair (shared memory, block scope) ---------------------------------
__device__ __forceinline__ int ld_acquire(const int* p) {
    int v;
    asm volatile("ld.acquire.cta.shared.s32 %0, [%1];" : "=r"(v) : "r"((unsigned)__cvta_generic_to_shared(p)) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
    asm volatile("st.release.cta.shared.s32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(p)), "r"(v) : "memory");
}

// position t of a producer's stream -> (cell c of the stream, sorted index ip of the particle, or ip = -1 for a pad
// position / the end of the stream).  cp[c] = first position of cell c (cp[NC] = length of the stream),
// off = the block's table of sorted indices at every cell boundary of every row.
template <class C>
__device__ __forceinline__ void stream_lookup(int t, const int* __restrict__ cp, const int* __restrict__ off_all,
                                              int row_first, int& c, int& ip) {
    int r = 0;
#pragma unroll
    for (int k = 1; k < C::RPW; ++k) r += (t >= cp[C::TX * k]);
    const int4 a = *reinterpret_cast<const int4*>(cp + C::TX * r), b = *reinterpret_cast<const int4*>(cp + C::TX * r + 4);
    const int q = (t >= a.y) + (t >= a.z) + (t >= a.w) + (t >= b.x) + (t >= b.y) + (t >= b.z) + (t >= b.w);
    c = C::TX * r + q;
    const int* off = off_all + (row_first + r) * (C::TX + 1) + q;
    const int lo = off[0], n = off[1] - lo, k = t - cp[c];
    ip = (t < cp[C::NC] && k < n) ? lo + k : -1;
}

// per-pair staging area
template <class C>
struct Staging {
    double* body;     // ring of record bodies
    double* tails;    // RING x (-q w / dt, e)
    int* codes;       // RING record codes
    double* scr;      // slow-path scratch record
    double* pbuf;     // landing buffer: [x y z ux uy uz w id][lane]
    int* cp;          // cp[NC + 1], 16-byte aligned
    int* flags;       // [0] = stream position up to which records are staged, [1] = ... consumed
    __device__ __forceinline__ explicit Staging(double* stg) {
        body = stg;
        tails = stg + C::BODY_W;
        codes = reinterpret_cast<int*>(tails + C::TAIL_W);
        scr = tails + C::TAIL_W + C::CODE_W + (C::CODE_W & 1);
        pbuf = scr + C::SLOW_W;
        cp = reinterpret_cast<int*>(pbuf + C::PBUF_W);
        flags = cp + ((C::NC + 1 + 3) & ~3);
    }
};

// ---- consumer warp: phase B and the flush of every row of its producer's stream -------------------------
// A producer does not wait for ring space for ever: after SPIN_LIMIT polls (seconds; a row takes microseconds) it sets
// bit 1 of the status flag, which the next synchronising call turns into a sticky PIC_ECUDA, publishes its whole stream
// as staged so that its consumer drains and leaves, and returns.  The consumer itself only ever waits for its producer,
// which always publishes the end of its stream (a guard inside the consumer's poll loop cost 4 % of the launch).
constexpr int SPIN_LIMIT = 1 << 24;

template <int N, class C>
__device__ __forceinline__ void tile_consumer(const Grid& g, const Fields& f, const Staging<C>& S, const int* row_off,
                                              int row_first, int t0x, int t0y, int t0z, int lane) {
    constexpr int FW = FastWin<N>::FW, FA = FastWin<N>::FA;
    const int* cp = S.cp;
    const int T = cp[C::NC];
    const double area_x = g.inv_dy * g.inv_dz, area_y = g.inv_dx * g.inv_dz, area_z = g.inv_dx * g.inv_dy;
    const int bq = lane >> 2, bs = lane & 3;     // cell of the row, plane of the window
    int b_lo = 0;                                // stream position up to which records have been consumed
    CellAcc<N> acc;
    acc.clear();
#pragma unroll 1
    for (int row_cur = 0; row_cur < C::RPW; ++row_cur) {
        const int row_lo = cp[C::TX * row_cur], row_end = cp[C::TX * (row_cur + 1)];
        if (row_end == row_lo) continue;         // empty row: nothing staged, nothing to flush
        const int row_t = row_first + row_cur;
        const long long win0 = g.idx(t0x + bq + FA, t0y + row_t % C::TY + FA, t0z + row_t / C::TY + FA);
        const int cs = cp[C::TX * row_cur + bq];
        const int ce = cs + (row_off[row_t * (C::TX + 1) + bq + 1] - row_off[row_t * (C::TX + 1) + bq]);
#pragma unroll 1
        for (;;) {
            // wait until the whole row is staged, or the producer has run out of ring space
            int staged;
            for (;;) {
                staged = ld_acquire(S.flags);
                if (staged >= row_end || (staged + C::AHEAD - b_lo > C::RING && staged < T)) break;
                __nanosleep(C::POLL_NS);      // a sub-chunk takes the producer ~6 us: polling faster only burns issue slots
            }
            const bool full_row = staged >= row_end;
            const int b_hi = full_row ? row_end : staged;
            {
                const int lo = max(cs, b_lo), hi = min(ce, b_hi);
                const int len = (bs < FW) ? hi - lo : 0;
                const int maxlen = __reduce_max_sync(0xffffffffu, max(len, 0));
                int sl = lo % C::RING;
#pragma unroll 1
                for (int t = 0; t < maxlen; ++t)
                    if (t < len) {
                        acc.add(S.body + body_word<C>(sl), ld2(S.tails, 2 * sl), S.codes[sl], bs, f.Jx + win0,
                                f.Jy + win0, f.Jz + win0, g.sy, g.sz, area_x, area_y, area_z);
                        sl = (sl + 1 == C::RING) ? 0 : sl + 1;
                    }
            }
            __syncwarp();
            b_lo = b_hi;
            if (lane == 0) st_release(S.flags + 1, b_lo);      // the slots below b_lo may be reused
            if (full_row) break;
        }
        acc.flush(g, f, win0, bs, lane);
        acc.clear();
    }
}

// ---- producer warp: phase A over its stream ------------------------------------------------------------
template <int N, int GV, class C>
__device__ __forceinline__ void tile_producer(const Grid& g, const Fields& f, const Particles& p, const Particles& po,
                                              const unsigned int* __restrict__ perm, unsigned int* __restrict__ key_out,
                                              double q, double h, const typename C::FT* __restrict__ Et, const Staging<C>& S,
                                              const int* row_off, int row_first, int t0x, int t0y, int t0z, int lane,
                                              DevStatus* status) {
    constexpr int FW = FastWin<N>::FW, FA = FastWin<N>::FA, DRIFT = C::DRIFT;
    using FR = FastRec<N>;
    using FT = typename C::FT;
    const int* cp = S.cp;
    double* pbuf = S.pbuf;
    const int T = cp[C::NC];
    if (T == 0) return;
    const double inv_c2 = 1.0 / (C_LIGHT * C_LIGHT);
    const double inv_dt = 1.0 / g.dt;
    unsigned int n_fast = 0, n_slow = 0, n_glob = 0;
    bool bad_any = false;

    // ---- software pipeline over the sub-chunks: lookup and perm[] two ahead, particle data one ahead --------
    int c0, ip0, c1, ip1, is1 = 0;
    stream_lookup<C>(lane, cp, row_off, row_first, c0, ip0);
    if (ip0 >= 0) {
        const int is = (perm != nullptr) ? (int)perm[ip0] : ip0;
        cp_async8(pbuf + 0 * 32 + lane, p.x + is); cp_async8(pbuf + 1 * 32 + lane, p.y + is);
        cp_async8(pbuf + 2 * 32 + lane, p.z + is); cp_async8(pbuf + 3 * 32 + lane, p.ux + is);
        cp_async8(pbuf + 4 * 32 + lane, p.uy + is); cp_async8(pbuf + 5 * 32 + lane, p.uz + is);
        cp_async8(pbuf + 6 * 32 + lane, p.w + is);
        if (perm != nullptr) cp_async8(pbuf + 7 * 32 + lane, p.id + is);
    }
    cp_async_commit();
    stream_lookup<C>(32 + lane, cp, row_off, row_first, c1, ip1);
    if (ip1 >= 0) is1 = (perm != nullptr) ? ld_u32_now(perm + ip1) : ip1;

#pragma unroll 1
    for (int t0 = 0; t0 < T; t0 += 32) {
        cp_async_wait_all();
        __syncwarp();
        const double x = pbuf[0 * 32 + lane], y = pbuf[1 * 32 + lane], z = pbuf[2 * 32 + lane];
        double ux = pbuf[3 * 32 + lane], uy = pbuf[4 * 32 + lane], uz = pbuf[5 * 32 + lane];
        const double wgt = pbuf[6 * 32 + lane], idv = pbuf[7 * 32 + lane];
        __syncwarp();       // every lane has read: the buffer may be refilled
        // ---- the next sub-chunk's particle data start their way to the landing buffer NOW, so that they
        // have this whole sub-chunk to arrive; the lookup (and perm[]) of the one after it goes into registers
        if (ip1 >= 0) {
            cp_async8(pbuf + 0 * 32 + lane, p.x + is1); cp_async8(pbuf + 1 * 32 + lane, p.y + is1);
            cp_async8(pbuf + 2 * 32 + lane, p.z + is1); cp_async8(pbuf + 3 * 32 + lane, p.ux + is1);
            cp_async8(pbuf + 4 * 32 + lane, p.uy + is1); cp_async8(pbuf + 5 * 32 + lane, p.uz + is1);
            cp_async8(pbuf + 6 * 32 + lane, p.w + is1);
            if (perm != nullptr) cp_async8(pbuf + 7 * 32 + lane, p.id + is1);
        }
        cp_async_commit();
        int c2, ip2, is2 = 0;
        stream_lookup<C>(t0 + 64 + lane, cp, row_off, row_first, c2, ip2);
        if (ip2 >= 0) is2 = (perm != nullptr) ? ld_u32_now(perm + ip2) : ip2;

        // ---- everything of this sub-chunk that does not touch the ring: gather, push, move, store ----
        const int ip = ip0;
        const int slot = (t0 + lane) % C::RING;
        bool is_slow = false, fast = false;
        double xi = 0.0, et = 0.0, ze = 0.0, xi1 = 0.0, et1 = 0.0, ze1 = 0.0, qw = 0.0;
        double wxn[N + 1], wyn[N + 1], wzn[N + 1];
        int ci = 0, cj = 0, ck = 0, fxn = 0, fyn = 0, fzn = 0;
        if (ip >= 0) {
            const int row_t = row_first + c0 / C::TX;                 // the listed cell: tile row, x position
            const int ry0 = row_t % C::TY, rz0 = row_t / C::TY, rx0 = c0 % C::TX;
            qw = q * wgt;
            if (perm != nullptr) {          // deferred sort: the other buffer gets every array, in sorted order
                po.w[ip] = wgt;
                po.id[ip] = (unsigned long long)__double_as_longlong(idv);
            }
            xi = (x - g.xmin) * g.inv_dx; et = (y - g.ymin) * g.inv_dy; ze = (z - g.zmin) * g.inv_dz;
            ci = __double2int_rd(xi); cj = __double2int_rd(et); ck = __double2int_rd(ze);
            const int rx = rel_cell<DRIFT>(ci, t0x, C::TX, g.nx), ry = rel_cell<DRIFT>(cj, t0y, C::TY, g.ny),
                      rz = rel_cell<DRIFT>(ck, t0z, C::TZ, g.nz);
            const bool in_tile = rx >= -DRIFT && rx <= C::TX - 1 + DRIFT && t0x + rx <= g.nx - 1 + DRIFT &&
                                 ry >= -DRIFT && ry <= C::TY - 1 + DRIFT && t0y + ry <= g.ny - 1 + DRIFT &&
                                 rz >= -DRIFT && rz <= C::TZ - 1 + DRIFT && t0z + rz <= g.nz - 1 + DRIFT;
            fxn = shape_weights<N>(xi, wxn); fyn = shape_weights<N>(et, wyn); fzn = shape_weights<N>(ze, wzn);
            FT eb[6];
            if (in_tile) {
                constexpr int NS = GatherOrders<N, GV>::NS;
                // from global node index to tile slot: slot = node - (t0 - GL) + image shift
                const int shx = (rx - (ci - t0x)) + C::GL - t0x, shy = (ry - (cj - t0y)) + C::GL - t0y,
                          shz = (rz - (ck - t0z)) + C::GL - t0z;
                {
                    // weights in the gather's arithmetic type (the fp64 nodal ones stay for the deposit record)
                    FT gxn[N + 1], gyn[N + 1], gzn[N + 1], wxs[NS + 1], wys[NS + 1], ws[NS + 1], wzs[N + 1];
#pragma unroll
                    for (int k = 0; k <= N; ++k) { gxn[k] = (FT)wxn[k]; gyn[k] = (FT)wyn[k]; gzn[k] = (FT)wzn[k]; }
                    const int fxs = shape_weights_t<NS, FT>(xi - 0.5, wxs) + shx, fys = shape_weights_t<NS, FT>(et - 0.5, wys) + shy,
                              fzs = shape_weights_t<NS, FT>(ze - 0.5, ws) + shz;
#pragma unroll
                    for (int k = 0; k <= N; ++k) wzs[k] = (k <= NS) ? ws[(k <= NS) ? k : 0] : FT(0);
                    gather6_part<N, GV, C>(Et, fxn + shx, fyn + shy, fzn + shz, fxs, fys, fzs, gxn, gyn, gzn, wxs, wys,
                                           wzs, eb);
                }
            } else {
                gather_global6<N, GV, FT>(g, f, xi, et, ze, eb);
                ++n_glob;
            }
            {       // Boris in FT (mixed precision: the momenta are doubles that hold floats)
                FT tx = (FT)ux, ty = (FT)uy, tz = (FT)uz;
                boris_push<FT>((FT)h, (FT)inv_c2, tx, ty, tz, eb[0], eb[1], eb[2], eb[3], eb[4], eb[5]);
                ux = (double)tx; uy = (double)ty; uz = (double)tz;
            }
            const double dtg = dt_over_gamma(g.dt, inv_c2, ux, uy, uz);
            const double x1 = x + dtg * ux, y1 = y + dtg * uy, z1 = z + dtg * uz;
            xi1 = (x1 - g.xmin) * g.inv_dx; et1 = (y1 - g.ymin) * g.inv_dy; ze1 = (z1 - g.zmin) * g.inv_dz;
            const bool bad = !(isfinite(x1) && isfinite(y1) && isfinite(z1)) || !(fabs(xi1 - xi) < 1.0) ||
                             !(fabs(et1 - et) < 1.0) || !(fabs(ze1 - ze) < 1.0);
            bad_any = bad_any || bad;
            const double xw = wrap1(x1, g.xmin, g.xmax, g.Lx, g.open_mask & 1), yw = wrap1(y1, g.ymin, g.ymax, g.Ly, g.open_mask & 2),
                         zw = wrap1(z1, g.zmin, g.zmax, g.Lz, g.open_mask & 4);
            po.x[ip] = xw;
            po.y[ip] = yw;
            po.z[ip] = zw;
            if (key_out != nullptr) {       // the next pic_sort's key (same formula as key_hist_kernel)
                const int ki = min(max(__double2int_rd((xw - g.xmin) * g.inv_dx), 0), g.nx - 1);
                const int kj = min(max(__double2int_rd((yw - g.ymin) * g.inv_dy), 0), g.ny - 1);
                const int kk = min(max(__double2int_rd((zw - g.zmin) * g.inv_dz), 0), g.nz - 1);
                key_out[ip] = (unsigned int)ki + (unsigned int)g.nx * ((unsigned int)kj + (unsigned int)g.ny * (unsigned int)kk);
            }
            po.ux[ip] = ux;
            po.uy[ip] = uy;
            po.uz[ip] = uz;
            // ---- classify: fast = stayed inside the cell the sort listed it in -------------
            const bool listed = in_tile && rx == rx0 && ry == ry0 && rz == rz0;   // the particle sits in the cell it is listed under
            const bool deposits = !bad && qw != 0.0;
            const int ncross = (__double2int_rd(xi1) != ci) + (__double2int_rd(et1) != cj) +
                               (__double2int_rd(ze1) != ck);
            fast = deposits && listed && ncross <= 1;   // phase B handles one crossed face
            is_slow = deposits && !fast;
            if (in_tile) { if (is_slow) ++n_slow; else ++n_fast; }
        }
        // ---- the ring slots of this sub-chunk must have been consumed ------------------------------
        for (int spins = 0; t0 + 32 - ld_acquire(S.flags + 1) > C::RING; ++spins) {
            if (spins > SPIN_LIMIT) {      // give up: flag the error and release the consumer (it drains stale slots)
                atomicOr(&status->ephys, 2);
                if (lane == 0) st_release(S.flags, T);
                return;
            }
            __nanosleep(32);
        }
        if (ip >= 0) {
            double* rec = S.body + body_word<C>(slot);
            if (fast) {
                // ---- fast record: old shapes and shape differences on the cell's window -------------
                double fr[FR::LEN];
                int code = REC_FAST;
                double ext_e = 0.0;
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const double a1 = (d == 0) ? xi1 : ((d == 1) ? et1 : ze1);
                    const int cell = (d == 0) ? ci : ((d == 1) ? cj : ck);
                    const int f0 = (d == 0) ? fxn : ((d == 1) ? fyn : fzn);
                    const double (&w0)[N + 1] = (d == 0) ? wxn : ((d == 1) ? wyn : wzn);
                    double w1[N + 1], s0[FW], s1[FW], e_lo, e_hi;
                    const int f1 = shape_weights<N>(a1, w1);
                    to_fast_window<N>(w0, f0, cell + FA, s0);
                    place_new_window<N>(w1, f1 - (cell + FA), s1, e_lo, e_hi);
#pragma unroll
                    for (int a = 0; a < FW - 1; ++a) {
                        fr[FR::s0(d, a)] = s0[a];
                        fr[FR::ds(d, a)] = s1[a] - s0[a];
                    }
                    if (e_lo != 0.0) { code = 1 + 2 * d; ext_e = e_lo; }
                    if (e_hi != 0.0) { code = 2 + 2 * d; ext_e = e_hi; }
                }
#pragma unroll
                for (int k = 0; k < FR::LEN / 2; ++k) st2(rec, 2 * k, fr[2 * k], fr[2 * k + 1]);
                st2(S.tails, 2 * slot, -qw * inv_dt, ext_e);
                S.codes[slot] = code;
            } else if (is_slow) {
                st2(rec, 0, xi, et); st2(rec, 2, ze, xi1); st2(rec, 4, et1, ze1); st2(rec, 6, qw, 0.0);
                S.codes[slot] = REC_SLOW;
            } else {
                S.codes[slot] = REC_NONE;
            }
        }
        __syncwarp();
        // ---------------- slow path: one particle at a time, whole warp ---------------------
        unsigned int slow_mask = __ballot_sync(0xffffffffu, is_slow);
        while (slow_mask) {
            const int L = __ffs(slow_mask) - 1;
            slow_mask &= slow_mask - 1;
            slow_build<N>(S.body + body_word<C>((t0 + L) % C::RING), S.scr, g, inv_dt, lane);
            slow_deposit<N>(S.scr, g, f, lane);
            __syncwarp();
        }
        // publish: the records up to here are staged (the consumer skips slow and empty slots by their code)
        if (lane == 0) st_release(S.flags, min(T, t0 + 32));
        c0 = c1; ip0 = ip1; c1 = c2; ip1 = ip2; is1 = is2;
    }
    // ---- flags and counters ----------------------------------------------------------------------
    if (bad_any) atomicOr(&status->ephys, 1);
    n_fast = __reduce_add_sync(0xffffffffu, n_fast);
    n_slow = __reduce_add_sync(0xffffffffu, n_slow);
    n_glob = __reduce_add_sync(0xffffffffu, n_glob);
    if (lane == 0) {
        if (n_fast) atomicAdd(&status->n_fast, (unsigned long long)n_fast);
        if (n_slow) atomicAdd(&status->n_slow, (unsigned long long)n_slow);
        if (n_glob) atomicAdd(&status->n_global, (unsigned long long)n_glob);
    }
}

template <int N, int GV, class C>
__global__ void __launch_bounds__(C::NT, C::MINB)
particles_tile_kernel(Grid g, Fields f, Particles p, Particles po, const unsigned int* __restrict__ perm,
                      unsigned int* __restrict__ key_out, double q, double h,
                      const unsigned int* __restrict__ cell_offset, int ntx, int nty, DevStatus* status) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using FT = typename C::FT;
    FT* Et = reinterpret_cast<FT*>(smem_raw);                    // TOT words of FT: Ex Ey Ez Bx By Bz
    double* stg_all = reinterpret_cast<double*>(smem_raw) + C::TOT_D;   // NP * STG_W
    int* row_off = reinterpret_cast<int*>(stg_all + C::NP * C::STG_W);   // NROW x (TX+1) container indices

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int b = blockIdx.x;
    const int bx = b % ntx; b /= ntx;
    const int by = b % nty;
    const int bz = b / nty;
    const int t0x = bx * C::TX, t0y = by * C::TY, t0z = bz * C::TZ;

    // ---- container index of every cell boundary of the tile's rows --------------------------
    for (int e = tid; e < C::NOFF; e += C::NT) {
        const int r = e / (C::TX + 1), c = e % (C::TX + 1);
        const int j = t0y + r % C::TY, k = t0z + r / C::TY;
        int v = 0;
        if (j < g.ny && k < g.nz)
            v = (int)cell_offset[(long long)g.nx * (j + (long long)g.ny * k) + min(t0x + c, g.nx)];
        row_off[e] = v;
    }
    __syncthreads();
    int n_tile = 0;
#pragma unroll 4
    for (int r = 0; r < C::NROW; ++r) n_tile += row_off[r * (C::TX + 1) + C::TX] - row_off[r * (C::TX + 1)];
    if (n_tile == 0) return;    // empty tile (block-uniform)

    // ---- stage the field stencil ----------------------------------------------------------------
    // All of a thread's loads are issued before the first store (one L2/HBM round trip instead of one
    // per loop trip).
    {
        const double* src[6] = {f.Ex, f.Ey, f.Ez, f.Bx, f.By, f.Bz};
        constexpr int NIT = (C::ESZ + C::NT - 1) / C::NT;
        double v[NIT][6];
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int e = tid + it * C::NT;
            const int ex = e % C::EX, ey = (e / C::EX) % C::EY, ez = e / (C::EX * C::EY);
            const int gx = t0x - C::GL + ex + NG, gy = t0y - C::GL + ey + NG, gz = t0z - C::GL + ez + NG;
            const bool ok = e < C::ESZ && gx >= 0 && gx < g.nx + 2 * NG && gy >= 0 && gy < g.py && gz >= 0 &&
                            gz < g.pz;
            const long long o = gx + g.sy * gy + g.sz * gz;
#pragma unroll
            for (int cpt = 0; cpt < 6; ++cpt) v[it][cpt] = ok ? __ldg(src[cpt] + o) : 0.0;
        }
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int e = tid + it * C::NT;
            if (e < C::ESZ) {
                const int w = tile_word<C>(e % C::EX, (e / C::EX) % C::EY, e / (C::EX * C::EY));
#pragma unroll
                for (int cpt = 0; cpt < 6; ++cpt)
                    if (!(C::trimmed(cpt) && e % C::EX == 0)) Et[C::comp_base(cpt) + w] = (FT)v[it][cpt];
            }
        }
    }

    // ---- a producer's stream: its RPW rows, cell by cell ---------------------------------------------------
    const int pair = (warp < C::NP) ? warp : warp - C::NP;
    const Staging<C> S(stg_all + pair * C::STG_W);
    const int row_first = pair * C::RPW;
    if (warp < C::NP) {
        int carry = 0;
#pragma unroll
        for (int half = 0; half < (C::NC + 31) / 32; ++half) {
            const int c = half * 32 + lane;
            int n = 0;
            if (c < C::NC) {
                const int* o = row_off + (row_first + c / C::TX) * (C::TX + 1) + c % C::TX;
                n = o[1] - o[0];
            }
            int incl = n;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += t;
            }
            if (c < C::NC) S.cp[c] = carry + incl - n;
            carry += __shfl_sync(0xffffffffu, incl, 31);
        }
        if (lane == 0) {
            S.cp[C::NC] = carry;
            S.flags[0] = 0;
            S.flags[1] = 0;
        }
    }
    __syncthreads();      // stencil, cp[] and the flags of every pair

    if (warp < C::NP)
        tile_producer<N, GV, C>(g, f, p, po, perm, key_out, q, h, Et, S, row_off, row_first, t0x, t0y, t0z, lane, status);
    else
        tile_consumer<N, C>(g, f, S, row_off, row_first, t0x, t0y, t0z, lane);
}

// CfgDrift: a species that has moved since its last sort (particles up to one cell outside their listed
// cell still gather from shared memory); one block of 6 + 6 warps per SM, tile 8 x 4 x 6.
// CfgFresh: right after pic_sort; two blocks of 3 + 3 warps per SM, tile 8 x 4 x 6.  Ring depth: 29.1 ms per launch with
// 120 slots, 30.1 with 104, 31.2 with 88 (rows of 64 +- 8 records plus the 31 a sub-chunk runs ahead stop fitting and
// are consumed in two passes); deeper than 120 buys nothing at 8 particles per cell (a 12-double record with the old
// shapes recomputed by the consumer and 168 slots: 29.4 ms).  (Measured and dropped,
// profiles/r02_tile_kernel.md: one consumer for two producers -- its duty is 56 % -- at 4 + 2 warps per block runs at
// 34.2 instead of 29.2 ms: decoupling two producers needs rings two rows deep, which shared memory does not have.)
// *32: the mixed-precision mode (fp32 stencil, gather and push; same tiles and rings).
using CfgDrift = TileCfg<8, 4, 6, 6, 1, 1, 112>;
using CfgFresh = TileCfg<8, 4, 6, 3, 2, 0, 120>;
using CfgDrift32 = TileCfg<8, 4, 6, 6, 1, 1, 112, float>;
using CfgFresh32 = TileCfg<8, 4, 6, 3, 2, 0, 120, float>;
static_assert(2 * (CfgFresh::SMEM + 1024) <= 228 * 1024, "two fresh-sort blocks must fit one SM");
static_assert(CfgDrift::SMEM <= 227 * 1024, "the drift block must fit one SM");

template <int N, int GV, class Cfg>
void launch_tile(const Grid& g, const Fields& f, const Particles& p, const Particles& po, const unsigned int* perm,
                 unsigned int* key_out, double q, double h, const unsigned int* cell_offset, DevStatus* status,
                 cudaStream_t st) {
    const int ntx = (g.nx + Cfg::TX - 1) / Cfg::TX, nty = (g.ny + Cfg::TY - 1) / Cfg::TY,
              ntz = (g.nz + Cfg::TZ - 1) / Cfg::TZ;
    const long long nb = (long long)ntx * nty * ntz;
    particles_tile_kernel<N, GV, Cfg><<<(unsigned)nb, Cfg::NT, Cfg::SMEM, st>>>(g, f, p, po, perm, key_out, q, h,
                                                                               cell_offset, ntx, nty, status);
}

template <int N, int GV, class Cfg>
cudaError_t setup_one() {
    cudaError_t e = cudaFuncSetAttribute(particles_tile_kernel<N, GV, Cfg>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)Cfg::SMEM);
    if (e == cudaSuccess && Cfg::MINB > 1)
        e = cudaFuncSetAttribute(particles_tile_kernel<N, GV, Cfg>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                 (int)cudaSharedmemCarveoutMaxShared);
    return e;
}

template <int GV, class Cfg>
cudaError_t setup_orders() {
    cudaError_t e = setup_one<1, GV, Cfg>();
    if (e == cudaSuccess) e = setup_one<2, GV, Cfg>();
    if (e == cudaSuccess) e = setup_one<3, GV, Cfg>();
    return e;
}

template <class Cfg>
cudaError_t setup_cfg() {
    cudaError_t e = setup_orders<0, Cfg>();
    if (e == cudaSuccess) e = setup_orders<1, Cfg>();
    return e;
}

template <int GV, class Cfg>
void launch_orders(int order, const Grid& g, const Fields& f, const Particles& p, const Particles& po,
                   const unsigned int* perm, unsigned int* key_out, double q, double h, const unsigned int* cell_offset,
                   DevStatus* status, cudaStream_t st) {
    if (order == 1) launch_tile<1, GV, Cfg>(g, f, p, po, perm, key_out, q, h, cell_offset, status, st);
    else if (order == 2) launch_tile<2, GV, Cfg>(g, f, p, po, perm, key_out, q, h, cell_offset, status, st);
    else launch_tile<3, GV, Cfg>(g, f, p, po, perm, key_out, q, h, cell_offset, status, st);
}

template <class Cfg>
void launch_cfg(int order, int gather_variant, const Grid& g, const Fields& f, const Particles& p, const Particles& po,
                const unsigned int* perm, unsigned int* key_out, double q, double h, const unsigned int* cell_offset,
                DevStatus* status, cudaStream_t st) {
    if (gather_variant) launch_orders<1, Cfg>(order, g, f, p, po, perm, key_out, q, h, cell_offset, status, st);
    else launch_orders<0, Cfg>(order, g, f, p, po, perm, key_out, q, h, cell_offset, status, st);
}

}  // namespace

int tile_setup() {
    cudaError_t e = setup_cfg<CfgDrift>();
    if (e == cudaSuccess) e = setup_cfg<CfgFresh>();
    if (e == cudaSuccess) e = setup_cfg<CfgDrift32>();
    if (e == cudaSuccess) e = setup_cfg<CfgFresh32>();
    return (int)e;
}

int launch_particles_tile(const Grid& g, const Fields& f, const Particles& p, const Particles& po,
                          const unsigned int* perm, unsigned int* key_out, long long n, double q, double m, int order,
                          int gather_variant, int precision, const unsigned int* cell_offset, bool fresh,
                          DevStatus* status, cudaStream_t st) {
    if (n <= 0) return 0;
    const double h = q * g.dt / (2.0 * m);
    if (precision) {
        if (fresh) launch_cfg<CfgFresh32>(order, gather_variant, g, f, p, po, perm, key_out, q, h, cell_offset, status, st);
        else launch_cfg<CfgDrift32>(order, gather_variant, g, f, p, po, perm, key_out, q, h, cell_offset, status, st);
    } else {
        if (fresh) launch_cfg<CfgFresh>(order, gather_variant, g, f, p, po, perm, key_out, q, h, cell_offset, status, st);
        else launch_cfg<CfgDrift>(order, gather_variant, g, f, p, po, perm, key_out, q, h, cell_offset, status, st);
    }
    return 1;
}

}  // namespace pic
