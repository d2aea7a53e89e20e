// Resident-tile kernel of the Shan-Chen models (sm_100a): ONE persistent, warp-specialised launch per time step in
// which every population crosses HBM once in each direction.
//
// The problem: Eq. 11 / 13 need psi(x + c_i, t) of all neighbours before cell x
// is collided (R9), and rho(x, t + 1) = sum_i f*_i(x - c_i, t) (Eq. 5 / 7) needs the step of all neighbours.  Two
// launches per time step (k_psi, k_step) read the flow populations twice from HBM.  Here the psi pass of time level
// t + 1 TRAILS the step of time level t inside the same launch, so that it reads the populations the step has just
// written while they are still in L2 (126 MB).  One block per SM works through the tickets b, b + B, ... of a
// host-built list (tile_schedule.h, path_setup); a ticket names a tile to step (its STEP part) and a tile whose
// psi(t + 1) is due (its PSI part), one tile = 1 KB rows (256 fp32 / 128 fp64 cells of an x-row):
//
//   producer warps  (4 for the STEP parts, 2 for the PSI parts, one 'landed' barrier per part and stage) The rows of a part
//                   into the next free stage of a ring of shared-memory stages -- one cp.async.bulk (TMA unit, UBLKCP;
//                   completion as transaction bytes on an mbarrier) per row, issued by the lane that owns the row.  STEP part: the S*Q + Q_s slot rows P_i(x) of the tile and the psi(t)
//                   rows around it (3 x 3 rows per component); at odd parity a population row comes from the neighbour
//                   row (y - c_y, z - c_z) and is shifted by -c_x: the aligned segment plus the 16-byte piece left or
//                   right of it (16-byte cp.async; also the one-cell halo of the psi rows).  PSI part: first the flags
//                   of the up to 27 tiles around the tile (acquire), then its S*Q flow rows at the NEXT parity.
//   step warps      (two teams of TX / cells-per-thread threads, both on every ticket, swapping parts) STEP part: steps
//                   a1, a3-a8 from the stage -- moments, psi stencil, force, collide, store to the global slots the rows
//                   came from; in fp32 every thread owns TWO cells and runs the packed f32x2 instantiation (V = F2) of
//                   the cell arithmetic.  PSI part: step a2 for t + 1 -- rho^sigma in index order (Eq. 7 / 18), psi^sigma
//                   (Eq. 10 / 24 or psi = rho) to the second psi buffer, which the next launch reads.
//   publisher warp  once all warps of a team have stored a STEP tile: one gpu-scope fence, then the tile's flag (launch
//                   epoch) in global memory.
//
// Deadlock freedom: a ticket depends only on the STEP parts of EARLIER tickets (its PSI part on the steps of the tiles
// around that tile; its STEP part on nothing), every block takes its tickets in list order, and the host launches at
// most as many blocks as are co-resident: the earliest unfinished ticket of the list can always proceed.  Every wait
// is bounded (clock64); a timeout sets bits in *status and gives up instead of hanging the GPU.
//
// Requirements (else the two-launch path runs): periodic x, nx * sizeof(R) a multiple of 16 bytes, no solid mask;
// either forcing scheme.  Walls in y / z are uniform per row and handled here: rows beyond a wall are redirected to the
// cell's own slot (halfway bounce-back) and left out of the psi stencil (Eq. 11-12), adhesion Eq. 14 and moving walls
// (moving_wall_rows) included.
#pragma once
#include "kernels.cuh"
#include "tile_schedule.h"

namespace lbm {

// bytes of one row segment of a tile (one bulk copy): a multiple of 16
#ifndef LBM_TILE_ROW_BYTES
#define LBM_TILE_ROW_BYTES 1024
#endif
constexpr int TILE_ROW_BYTES = LBM_TILE_ROW_BYTES;
// producer warps per block: for the STEP parts (they never wait for another block) and for the PSI parts (they wait for
// the flags of the tiles around the PSI tile); each lane looks after one row
#ifndef LBM_TILE_PRODS
#define LBM_TILE_PRODS 4
#endif
#ifndef LBM_TILE_PRODP
#define LBM_TILE_PRODP 2
#endif

// (struct TileItem, one ticket: tile_schedule.h)
struct TilePos {
    int xs, y, z;
};

struct TileArgs {
    const TileItem* items;            // the tickets of one time step (device): a tile to step and / or a tile whose psi is due
    unsigned n_items;                 // tickets (tiles + the tail of PSI-only tickets)
    int nxs;                          // tiles per row
    int* flags;                       // one per tile (z, y, xs): launch epoch of the last completed step
    int epoch;                        // > 0, differs from every earlier launch since the flags were cleared
    int* status;                      // bits set when a bounded wait timed out
    void* psi_out;                    // psi(t + 1): S * N values, not the buffer KP::psi points at
    int moving;                       // some wall in y / z has a velocity (KP::wall_u): moving-wall bounce-back on the edge rows
#ifdef LBM_TILE_TRACE
    long long* trace;
#endif
};

#ifdef LBM_TILE_TRACE
// developer trace: time stamps of block 0's roles per ticket (0 copies issued, 1 stage full seen by the step warps,
// 2 flag published, 3 flags seen by psi warp 0, 4 psi stored, 5 step start, 6 step end, 7 free stage seen by the producer)
__device__ __forceinline__ void tile_trace(long long* buf, int what, unsigned n) {
    if (blockIdx.x == 0 && (threadIdx.x & 31) == 0 && n < 4096) {
        long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        buf[what * 4096 + n] = t;
    }
}
#define TILE_TRACE(what, n) tile_trace(w.trace, what, n)
#else
#define TILE_TRACE(what, n)
#endif

// ---- PTX helpers ----
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
// (LDG.STRONG.GPU + CCTL.IVALL: no MEMBAR, unlike a relaxed load followed by fence.acq_rel.gpu, which waits for the
// warp's own outstanding stores)
__device__ __forceinline__ int ld_acquire(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ int ld_relaxed(const int* p) {
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_relaxed(int* p, int v) {
    asm volatile("st.relaxed.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ unsigned ld_acquire_cta_shared(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.cta.shared::cta.u32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_cta_shared(unsigned* p, unsigned v) {
    asm volatile("st.release.cta.shared::cta.u32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// (the suspend-time hint lets a waiting warp sleep in hardware instead of spinning on its scheduler's issue slots)
constexpr unsigned TILE_SUSPEND_NS = 20000u;
__device__ __forceinline__ bool mbar_try_wait(unsigned long long* bar, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity), "r"(TILE_SUSPEND_NS)
        : "memory");
    return ok != 0;
}
constexpr long long TILE_TIMEOUT_CYCLES = 6000000000LL;     // ~3 s: far beyond any legitimate wait
// bounded wait for the phase with the given parity; false (and *status |= code) on timeout
__device__ __forceinline__ bool mbar_wait(unsigned long long* bar, unsigned parity, int* status, int code) {
    if (mbar_try_wait(bar, parity)) return true;
    const long long t0 = clock64();
    while (!mbar_try_wait(bar, parity)) {
        if (clock64() - t0 > TILE_TIMEOUT_CYCLES) { atomicOr(status, code); return false; }
    }
    return true;
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// global -> shared bulk copy by the TMA unit (bytes a multiple of 16, both addresses 16-byte aligned), completion
// counted as transaction bytes on bar
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// the same with an L2 eviction policy (createpolicy): populations are read once per launch -- evict_first keeps L2 for
// the lines the step WRITES, which the trailing psi tickets read back
__device__ __forceinline__ unsigned long long l2_evict_first() {
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void bulk_g2s_hint(unsigned dst, const void* src, unsigned bytes, unsigned long long* bar, unsigned long long pol) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
                 : "memory");
}
// 16-byte asynchronous copy global -> shared (LDGSTS.128, L2 only) and its completion on an mbarrier: the barrier
// receives one arrival from the executing thread once all its earlier cp.async have landed (.noinc: the arrival is
// part of the barrier's initial count)
// (no "memory" clobber: ordinary loads of the row tables may be scheduled across the copies; ordering against the
// consumers comes from the mbarrier operations, which do clobber memory)
__device__ __forceinline__ void cp_async16(unsigned dst, const void* src) {
#ifdef LBM_TILE_CA
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src));
#else
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src));
#endif
}
__device__ __forceinline__ void cp_async_arrive(unsigned long long* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// stores through an address read from shared memory: say "global" (a generic ST would check the address space)
__device__ __forceinline__ void st_global(float* p, float v) { asm volatile("st.global.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory"); }
__device__ __forceinline__ void st_global(double* p, double v) { asm volatile("st.global.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory"); }
__device__ __forceinline__ void st_global(float* p, F2 v) { asm volatile("st.global.b64 [%0], %1;" ::"l"(p), "l"(v.v) : "memory"); }

// c_{i,a} for a RUN-TIME i without a table in local memory: two bits per direction in a compile-time word
template <class LL>
__host__ __device__ constexpr unsigned long long packed_axis(int a) {
    unsigned long long v = 0;
    for (int i = 0; i < LL::Q; ++i) v |= (unsigned long long)(LL::c(i, a) + 1) << (2 * i);
    return v;
}
template <class LL, int A>
__device__ __forceinline__ int c_runtime(int i) {
    constexpr unsigned long long pk = packed_axis<LL>(A);
    return (int)((pk >> (2 * i)) & 3ULL) - 1;
}

// One block per SM (__launch_bounds__(THREADS, 1)): the stages fill the shared memory, the warps the register file.
template <class R, class L, int MODEL>
struct TileCfg {
    using MT = ModelTraits<MODEL>;
    using LS = typename ScalarOf<L>::type;
    static constexpr bool PACK = sizeof(R) == 4;                 // two fp32 cells per step thread, packed arithmetic
    using V = std::conditional_t<PACK, F2, R>;
    static constexpr int CPT = PACK ? 2 : 1;
    static constexpr int S = MT::S, Q = L::Q, D = L::D;
    static constexpr int B = (int)sizeof(R);
    static constexpr int TX = TILE_ROW_BYTES / B;                // cells per tile
    static constexpr int H = 16 / B;                             // elements per 16-byte piece = halo width
    static constexpr int RS = TX + 2 * H;                        // elements per shared-memory row: [piece | segment | piece]
    static constexpr int NF = S * Q;
    static constexpr int NH = MT::SCALAR ? LS::Q : 0;
    static constexpr int NPOPS = NF + NH;
    static constexpr int NPSI = D == 3 ? 9 : 3;                  // psi rows (dy, dz) per component
    static constexpr int NP = S * NPSI;
    static constexpr int NROWS = NPOPS + NP;                     // rows of a stage: populations, then psi
    static constexpr int STEP_WARPS = (TX / CPT + 31) / 32;
    static constexpr int STEP_THREADS = 32 * STEP_WARPS;        // (threads beyond the tile's cells idle)
    // Two teams of step warps work on two stages at a time (two warps per scheduler hide each other's latencies).  The
    // step role of the D3Q19 models in fp64 needs more registers (19 doubles per component and thread): one team.
    static constexpr bool HEAVY = B == 8 && Q > 9;
    static constexpr int TEAMS = HEAVY ? 1 : 2;
    static constexpr int PROD_S = HEAVY ? 2 : LBM_TILE_PRODS, PROD_P = LBM_TILE_PRODP;
    static constexpr int AUX_WARPS = 1 + PROD_S + PROD_P;                 // publisher, producers
    static constexpr int THREADS = 32 * AUX_WARPS + TEAMS * STEP_THREADS;
    static constexpr int SROWS = NROWS + NF;                     // a stage: the STEP part's rows, then the flow rows of the PSI part
    static constexpr size_t STAGE_BYTES = (size_t)SROWS * RS * B;
    // a ring of NS stages; a ticket brings a tile to step AND a tile whose psi(t + 1) is due, so that the fixed costs of
    // a stage (issue of the copies, HBM latency, hand-over) are paid once for both
    static constexpr int NS = (215 * 1024) / STAGE_BYTES >= 4 ? 4 : (int)((215 * 1024) / STAGE_BYTES);   // stages
    static constexpr size_t ROWPTR_BYTES = (size_t)NS * 128 * sizeof(unsigned long long);   // pointers of the (up to 128) rows of a stage
    static constexpr size_t ROWSX_BYTES = (size_t)NS * 128 * sizeof(int);
    static constexpr int NBAR = 3 * NS;                          // per stage: STEP part landed, PSI part landed, stage free
    static constexpr size_t SMEM = NS * STAGE_BYTES + ROWPTR_BYTES + ROWSX_BYTES + NBAR * 8 + 32;
    static_assert(NROWS <= 32 * PROD_S && NF <= 32 * PROD_P, "one row per producer lane");
    static_assert(TEAMS * STEP_WARPS <= 8, "done counters");
    static_assert(NS >= 2 && SMEM <= 227 * 1024, "shared memory");
    __host__ __device__ static constexpr int psi_row(int t, int cy, int cz) { return NPOPS + t * NPSI + (cy + 1) + (D == 3 ? 3 * (cz + 1) : 0); }
};

template <class R, class L, int MODEL, int PARITY, bool WALLYZ, bool VSHIFT = false>
struct Tile {
    using C = TileCfg<R, L, MODEL>;
    using MT = typename C::MT;
    using LS = typename C::LS;
    using V = typename C::V;
    static constexpr int S = C::S, Q = C::Q, D = C::D, B = C::B, H = C::H, RS = C::RS, NF = C::NF, NPOPS = C::NPOPS, CPT = C::CPT;
    static constexpr int NROWS = C::NROWS, SROWS = C::SROWS, NS = C::NS, TILE_TX = C::TX;

    const KP<R>& p;
    const TileArgs& w;
    R* stages;                          // [NS][SROWS][RS]
    unsigned long long* rowptr;         // [NS][128]: global address of element x = 0 of the row staged there (0: none)
    int* rowsx;                         // [NS][128]: its x-shift (-1, 0, +1): cell x reads position H + (x - x0) + shift
    unsigned long long *full, *empty;
    unsigned* done;                     // [TEAMS * STEP_WARPS]: tickets of its team that step warp k has stored

    __device__ __forceinline__ Tile(const KP<R>& kp, const TileArgs& wa, unsigned char* smem) : p(kp), w(wa) {
        stages = (R*)smem;
        rowptr = (unsigned long long*)(smem + NS * C::STAGE_BYTES);
        rowsx = (int*)((unsigned char*)rowptr + C::ROWPTR_BYTES);
        full = (unsigned long long*)((unsigned char*)rowsx + C::ROWSX_BYTES);
        empty = full + 2 * NS;                              // full[2 * stage + part] (part 0: STEP rows, 1: PSI rows), empty[stage]
        done = (unsigned*)(empty + NS);
    }
    __device__ __forceinline__ R* slot_base(int stage) const {
        return stages + (size_t)stage * SROWS * RS;
    }
    static __device__ __forceinline__ int wrap(int v, int n) { return v < 0 ? v + n : (v >= n ? v - n : v); }
    __device__ __forceinline__ bool wall_y() const { return WALLYZ && p.bc[1]; }
    __device__ __forceinline__ bool wall_z() const { return WALLYZ && D == 3 && p.bc[2]; }
    // does the row offset (dy, dz) from row (y, z) cross a bounce-back wall?
    __device__ __forceinline__ bool crosses(int y, int z, int dy, int dz) const {
        if constexpr (!WALLYZ) return false;
        return (wall_y() && (y + dy < 0 || y + dy >= p.ny)) || (wall_z() && (z + dz < 0 || z + dz >= p.nz));
    }
    __device__ __forceinline__ bool edge_row(int y, int z) const {
        return WALLYZ && ((wall_y() && (y == 0 || y == p.ny - 1)) || (wall_z() && (z == 0 || z == p.nz - 1)));
    }
    static __device__ __forceinline__ TileItem item_of(const TileItem* items, unsigned ticket) {
        const int4 a = __ldg((const int4*)(items + ticket)), b = __ldg((const int4*)(items + ticket) + 1);
        return TileItem{a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
    }
    __device__ __forceinline__ int* flag_of(int xs, int y, int z) const {
        const int nm = D == 3 ? p.ny : 1;
        const int ms = D == 3 ? y : 0, ss = D == 3 ? z : y;
        return w.flags + ((size_t)ss * nm + ms) * w.nxs + xs;
    }

    // ---------------- producer ----------------
    // The flag this lane looks at for a PSI ticket at (xs, y, z): lane l < 27 has one of the (up to) 27 tiles around it
    // (nullptr: no such tile beyond a wall, or lane >= 27)
    __device__ __forceinline__ const int* flag_around(const TilePos& it) const {
        const int l = (int)(threadIdx.x & 31);
        const int nm = D == 3 ? p.ny : 1, ns = D == 3 ? p.nz : p.ny;
        const int m = D == 3 ? it.y : 0, s = D == 3 ? it.z : it.y;
        const bool wm = D == 3 ? wall_y() : false, wsl = D == 3 ? wall_z() : wall_y();
        if (l >= 27) return nullptr;
        const int dx = l % 3 - 1, dm = (l / 3) % 3 - 1, ds = l / 9 - 1;
        int mm = m + dm, ss = s + ds;
        if ((wm && (mm < 0 || mm >= nm)) || (wsl && (ss < 0 || ss >= ns)) || (D == 2 && dm != 0)) return nullptr;
        mm = wrap(mm, nm); ss = wrap(ss, ns);
        return w.flags + ((size_t)ss * nm + mm) * w.nxs + wrap(it.xs + dx, w.nxs);
    }
    // wait until the step of the tiles around a PSI ticket is complete.  seen: the value a relaxed load of the lane's
    // flag returned one ticket earlier (the load's latency is hidden behind the previous ticket).  Once every lane has
    // SEEN the epoch, the copies issued afterwards read what was published before the flags: they are issued after the
    // loads have returned and read L2, where the publisher's fence has made the populations visible.  Otherwise: poll
    // with acquire loads.
    __device__ __forceinline__ bool wait_flags(const int* fl, int seen) const {
        bool ok = fl == nullptr || seen == w.epoch;
        if (!__all_sync(0xffffffffu, ok)) {
            if (!ok) {
                const long long t0 = clock64();
                while (!(ok = (ld_acquire(fl) == w.epoch))) {
                    __nanosleep(200);
                    if (clock64() - t0 > TILE_TIMEOUT_CYCLES) { atomicOr(w.status, 8); break; }
                }
            }
            ok = __all_sync(0xffffffffu, ok);              // (a warp barrier: every lane's copies come after every lane's acquire)
        }
        return ok;
    }
    // Row r of a ticket of kind K at parity PAR (STEP: the parity of this launch, all rows; PSI: the next parity, the
    // flow populations only): where it comes from relative to the ticket's row.  nbr: element 0 of row (0, 0) of the
    // source array / slot; own: the same for the cell's own slot (a population row that would cross a wall; a psi row is
    // left out)
    struct RowDesc {
        const R* nbr;
        const R* own;
        int dy, dz, sx;
    };
    __device__ __forceinline__ RowDesc row_desc(int r, int par, bool psi_ticket) const {
        const size_t N = (size_t)p.N;
        RowDesc d{nullptr, nullptr, 0, 0, 0};
        if (r < NPOPS && !(psi_ticket && r >= NF)) {
            int i, c0, c1, c2, op;
            const R* arr;
            if (r < NF) {
                const int s = r / Q;
                i = r - s * Q;
                arr = p.f + (size_t)s * Q * N;
                c0 = c_runtime<L, 0>(i); c1 = c_runtime<L, 1>(i); c2 = D == 3 ? c_runtime<L, 2>(i) : 0; op = L::opp(i);
            } else {
                i = r - NF;
                arr = p.h;
                c0 = c_runtime<LS, 0>(i); c1 = c_runtime<LS, 1>(i); c2 = D == 3 ? c_runtime<LS, 2>(i) : 0; op = LS::opp(i);
            }
            d.own = arr + (size_t)i * N;
            d.nbr = d.own;
            if (par == 1 && i != 0) {          // P_i(x) = slot opp(i) of cell x - c_i; beyond a wall: slot i of x itself
                d.nbr = arr + (size_t)op * N; d.dy = -c1; d.dz = -c2; d.sx = -c0;
            }
        } else if (r >= NPOPS && r < NROWS && !psi_ticket) {
            const int q0 = r - NPOPS, t = q0 / C::NPSI, q = q0 - t * C::NPSI;
            d.dy = D == 3 ? q % 3 - 1 : q - 1; d.dz = D == 3 ? q / 3 - 1 : 0;
            d.nbr = p.psi + (size_t)t * N;
        }
        return d;
    }
    // Producer warp `pw` of the `nw` warps of part PART (0: the STEP part of every ticket, rows 0 .. NROWS-1 of a stage; 1: the
    // PSI part, rows NROWS .. SROWS-1) looks after the rows pw + nw * lane of its part.  The STEP producers never wait
    // for another block; the PSI producers wait for the flags of the tiles around the PSI tile first.
    template <int PART>
    __device__ __forceinline__ void produce(int pw, int nw, unsigned n_mine, unsigned b0, unsigned stride) const {
        const int lane = (int)(threadIdx.x & 31);
        const int q = pw + nw * lane;                          // row within the part
        const int r = PART == 0 ? (q < NROWS ? q : SROWS) : (q < NF ? NROWS + q : SROWS);      // row of the stage (SROWS: none)
        const RowDesc d = PART == 1 ? row_desc(q, 1 - PARITY, true) : row_desc(q, PARITY, false);
        const unsigned long long pol = l2_evict_first();
        // the ticket after the current one and the flag value of its PSI part are loaded one ticket ahead
        const TileItem none{0, 0, 0, 0, 0, 0, 0, 0};
        TileItem nxt = n_mine > 0 ? item_of(w.items, b0) : none;
        const int* nfl = (PART == 1 && nxt.pv) ? flag_around(TilePos{nxt.px, nxt.py, nxt.pz}) : nullptr;
        int nseen = nfl ? ld_relaxed(nfl) : 0;
        for (unsigned n = 0; n < n_mine; ++n) {
            const TileItem it = nxt;
            const int* fl = nfl;
            const int seen = nseen;
            if (n + 1 < n_mine) {
                nxt = item_of(w.items, b0 + (n + 1) * stride);
                nfl = (PART == 1 && nxt.pv) ? flag_around(TilePos{nxt.px, nxt.py, nxt.pz}) : nullptr;
                nseen = nfl ? ld_relaxed(nfl) : 0;
            }
            const int stage = (int)(n % NS);
            const unsigned ph = (n / NS) & 1u;
            unsigned long long* fb = &full[2 * stage + PART];
            // the PSI part reads what the step of the tiles around its tile has written: it is listed well after them
            // (tile_schedule.h), so this wait is mostly a formality -- but it is what makes the read correct
            if (PART == 1 && it.pv && !wait_flags(fl, seen)) return;
            if (!mbar_wait(&empty[stage], ph ^ 1u, w.status, 2)) return;
            if (PART == 0 && pw == 0) TILE_TRACE(7, n);
            const bool have = PART == 1 ? it.pv != 0 : it.sv != 0;
            const int xs = PART == 1 ? it.px : it.sx, y = PART == 1 ? it.py : it.sy, z = PART == 1 ? it.pz : it.sz;
            const int x0 = xs * TILE_TX;
            const int len = min(TILE_TX, p.nx - x0);
            const R* src = nullptr;
            int sx = 0;
            if (r < SROWS) {
                if (have) {
                    if (crosses(y, z, d.dy, d.dz)) {
                        if (d.own) src = d.own + ((size_t)z * p.ny + y) * (size_t)p.nx;
                    } else if (d.nbr) {
                        const int yy = wrap(y + d.dy, p.ny), zz = D == 3 ? wrap(z + d.dz, p.nz) : 0;
                        src = d.nbr + ((size_t)zz * p.ny + yy) * (size_t)p.nx;
                        sx = d.sx;
                    }
                }
                rowptr[stage * 128 + r] = (unsigned long long)src;
                rowsx[stage * 128 + r] = sx;
            }
            // One cp.async.bulk (TMA unit, UBLKCP: no load/store-unit slots) per row for the segment, issued by the lane
            // that owns the row; completion: transaction bytes on the part's barrier.  The 16-byte pieces beside the
            // segment (periodic wrap in x) are 16-byte cp.async; the barrier also counts one arrival per lane for them.
            const bool halo_row = PART == 0 && r >= NPOPS && r < NROWS;     // a psi(t) row: one-cell halo on both sides
            const unsigned dst = smem_u32(slot_base(stage) + (size_t)(r < SROWS ? r : 0) * RS);
            const unsigned bytes = __reduce_add_sync(0xffffffffu, src ? (unsigned)(len * B) : 0u);
            if (lane == 0) mbar_arrive_expect_tx(fb, bytes);
            __syncwarp();
            if (src) {
#ifndef LBM_TILE_NOHINT
                if (!halo_row) bulk_g2s_hint(dst + (unsigned)(H * B), src + x0, (unsigned)(len * B), fb, pol);
                else
#endif
                bulk_g2s(dst + (unsigned)(H * B), src + x0, (unsigned)(len * B), fb);
                if (sx < 0 || halo_row) cp_async16(dst, src + (x0 == 0 ? p.nx - H : x0 - H));
                if (sx > 0 || halo_row) cp_async16(dst + (unsigned)((H + len) * B), src + (x0 + len == p.nx ? 0 : x0 + len));
            }
            cp_async_arrive(fb);
            if (PART == 0 && pw == 0) TILE_TRACE(0, n);
        }
    }

    // ---------------- reading a stage ----------------
    // population I of lattice LL (rows R0 ...) of the thread's cell(s); sb: position of the first cell in row 0 of the stage.
    // EDGE: the item touches a bounce-back wall, rows may have been redirected (shift from the table)
    template <class LL, int R0, int I, bool EDGE, int PAR = PARITY>
    __device__ __forceinline__ V read_pop(const R* sb, int stage) const {
        const R* q = sb + (R0 + I) * RS;
        if constexpr (PAR == 0 || I == 0 || LL::c(I, 0) == 0) {
            if constexpr (C::PACK) { F2 v; v.v = *reinterpret_cast<const unsigned long long*>(q); return v; }
            else return *q;
        } else {
            int sh = -LL::c(I, 0);
            if constexpr (EDGE) sh = rowsx[stage * 128 + R0 + I];
            if constexpr (C::PACK) return pack2(q[sh], q[sh + 1]);
            else return q[sh];
        }
    }
    template <class LL, int R0, bool EDGE, int PAR = PARITY>
    __device__ __forceinline__ void read_pops(const R* sb, int stage, V* fl) const {
        static_for<0, LL::Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            fl[i] = read_pop<LL, R0, i, EDGE, PAR>(sb, stage);
        });
    }

    // ---------------- step warps ----------------
    // f*_{opp(i)} back to P_i(x): the global row the stage row came from, column x + shift (periodic wrap).
    // col[0..3] = x - 1, x, x + 1, x + 2 with wrap (x + 1 only for the second cell of a packed pair)
    template <class LL, int R0, int I, bool EDGE>
    __device__ __forceinline__ void write_pop(int stage, const int* col, V val) const {
        R* g0 = (R*)rowptr[stage * 128 + R0 + I];
        if constexpr (PARITY == 0 || I == 0 || LL::c(I, 0) == 0) {
            st_global(g0 + col[1], val);
        } else {
            int sh = -LL::c(I, 0);
            if constexpr (EDGE) sh = rowsx[stage * 128 + R0 + I];
            if constexpr (C::PACK) {
                if (EDGE && sh == 0) {
                    st_global(g0 + col[1], val);
                } else {
                    float lo, hi;
                    unpack2(val, lo, hi);
                    st_global(g0 + col[1 + sh], lo);
                    st_global(g0 + col[2 + sh], hi);
                }
            } else {
                st_global(g0 + col[1 + sh], val);
            }
        }
    }
    template <class LL, int R0, bool EDGE>
    __device__ __forceinline__ void write_pops(int stage, const int* col, const V* fl) const {
        static_for<0, LL::Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            write_pop<LL, R0, i, EDGE>(stage, col, fl[LL::opp(i)]);
        });
    }
    // psi(t) of the thread's cell(s) at offset (CX, CY, CZ) from the psi rows of the stage; sb as in read_pop
    template <int CX, int CY, int CZ>
    __device__ __forceinline__ V psi_at(const R* sb, int t) const {
        const R* q = sb + C::psi_row(t, CY, CZ) * RS + CX;
        if constexpr (C::PACK) {
            if constexpr (CX == 0) { F2 v; v.v = *reinterpret_cast<const unsigned long long*>(q); return v; }
            else return pack2(q[0], q[1]);
        } else {
            return *q;
        }
    }
    // Moving-wall halfway bounce-back on a row next to a wall in y / z (DESIGN R24; moving_wall_correction
    // of kernels.cuh with the row-uniform wall test): a post-collision population f*_k that leaves through a wall comes
    // back minus 2 w_k rho^s (c_k . u_w) / c_s^2; a direction crossing two walls takes the y wall
    __device__ __forceinline__ void moving_wall_rows(const TilePos& it, V rho_s, V* fl) const {
        static_for<1, Q>([&](auto kc) {
            constexpr int k = decltype(kc)::value;
            constexpr int CY = L::c(k, 1), CZ = L::c(k, 2);
            if constexpr (CY != 0 || CZ != 0) {
                if (crosses(it.y, it.z, CY, CZ)) {
                    const R* uw = nullptr;
                    if constexpr (CY != 0) { if (wall_y() && (CY < 0 ? it.y == 0 : it.y == p.ny - 1)) uw = p.wall_u[1][CY < 0 ? 0 : 1]; }
                    if constexpr (CZ != 0) { if (!uw && wall_z() && (CZ < 0 ? it.z == 0 : it.z == p.nz - 1)) uw = p.wall_u[2][CZ < 0 ? 0 : 1]; }
                    const R u3[3] = {uw[0], uw[1], uw[2]};
                    const R cuw = dotc<L, k>(u3);
                    fl[k] = vfma(-(vconst<V>(6.0 * L::w(k)) * rho_s), vbcast<V>(cuw), fl[k]);
                }
            }
        });
    }
    template <bool EDGE>
    __device__ __forceinline__ void step_cells(int stage, const TilePos& it, int t) const {
        const int x = it.xs * TILE_TX + t;
        const R* sb = slot_base(stage) + H + t;
        // The populations are read from the stage twice -- for the moments here, for the collision below -- instead of
        // being kept in registers in between (2 x 19 + 7 values per cell, two cells per thread): the step role then fits
        // 128 registers, which buys a second team of step warps per SM.  Same values, same arithmetic.
        CellMacro<V, L, MODEL> m;
        static_for<0, S>([&](auto sc) {
            constexpr int s = decltype(sc)::value;
            V fl[Q];
            read_pops<L, s * Q, EDGE>(sb, stage, fl);
            m.j[s][0] = m.j[s][1] = m.j[s][2] = vconst<V>(0.0);
            moments<L>(fl, m.rho[s], m.j[s]);
        });
        asm volatile("" ::: "memory");                     // (the second read below is a real read)

        // stencil sums from the psi rows, the order of sc_stencil (row a3)
        V acc[S][3], psi_own[S], adh[3];
        adh[0] = adh[1] = adh[2] = vconst<V>(0.0);
        static_for<0, S>([&](auto tc) {
            constexpr int tt = decltype(tc)::value;
            acc[tt][0] = acc[tt][1] = acc[tt][2] = vconst<V>(0.0);
            static_for<1, Q>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                constexpr int CX = L::c(i, 0), CY = L::c(i, 1), CZ = L::c(i, 2);
                bool out = false;
                if constexpr (EDGE) out = crosses(it.y, it.z, CY, CZ);
                V pv = vconst<V>(0.0);
                if (!out) pv = psi_at<CX, CY, CZ>(sb, tt);
                static_for<0, D>([&](auto ac) {
                    constexpr int a = decltype(ac)::value;
                    constexpr int c = L::c(i, a);
                    if constexpr (c != 0) {
                        acc[tt][a] = vfma(vconst<V>(c * L::w(i)), pv, acc[tt][a]);
                        if constexpr (EDGE && tt == 0) {      // adh_a = sum_{i>=1, solid neighbour} c_{i,a} w_i: Eq. 14
                            if (out) adh[a] = adh[a] + vconst<V>(c * L::w(i));
                        }
                    }
                });
            });
            psi_own[tt] = psi_at<0, 0, 0>(sb, tt);
        });
        cell_force_velocity<V, L, MODEL, true, WALLYZ>(p, acc, psi_own, m, adh);
        const int col[4] = {x == 0 ? p.nx - 1 : x - 1, x, x + 1 == p.nx ? 0 : x + 1, x + 2 >= p.nx ? x + 2 - p.nx : x + 2};
        V ueq[S][3];                                       // velocity-shift forcing scheme (Eq. 16-19): no forcing term F_i
        if constexpr (VSHIFT) shift_velocities<V, L, MODEL>(p, m, ueq);
        static_for<0, S>([&](auto sc) {
            constexpr int s = decltype(sc)::value;
            V fl[Q];
            read_pops<L, s * Q, EDGE>(sb, stage, fl);
            if constexpr (VSHIFT) collide_component<V, L, false, s>(p, fl, m.rho[s], ueq[s], m.F[s]);
            else collide_component<V, L, true, s>(p, fl, m.rho[s], m.u, m.F[s]);
            if constexpr (EDGE) {
                if (w.moving) moving_wall_rows(it, m.rho[s], fl);
            }
            write_pops<L, s * Q, EDGE>(stage, col, fl);
        });
        if constexpr (MT::SCALAR) {
            V hl[LS::Q];
            read_pops<LS, NF, EDGE>(sb, stage, hl);
            collide_scalar<V, LS>(p, hl, m.rho[0], m.rho[S - 1], m.inv_rho, m.u);
            write_pops<LS, NF, EDGE>(stage, col, hl);
        }
    }
    // step a2 for time level t + 1 (the PSI part of a ticket): rho^sigma in index order (Eq. 7 / 18) from the flow
    // populations the stage holds at the NEXT parity (rows NROWS ...), psi^sigma (Eq. 10 / 24 or psi = rho) to the second
    // psi buffer
    template <bool EDGE>
    __device__ __forceinline__ void psi_cells(int stage, const TilePos& it, int t) const {
        const R* sb = slot_base(stage) + H + t;
        R* out = (R*)w.psi_out + ((size_t)it.z * p.ny + it.y) * (size_t)p.nx + (it.xs * TILE_TX + t);
        static_for<0, S>([&](auto sc) {
            constexpr int s = decltype(sc)::value;
            V fl[Q];
            read_pops<L, NROWS + s * Q, EDGE, 1 - PARITY>(sb, stage, fl);
            V rho = fl[0];
            static_for<1, Q>([&](auto ic) { rho = rho + fl[decltype(ic)::value]; });
            st_global(out + (size_t)s * (size_t)p.N, psi_of(rho, p.psi_kind, p.rho0_psi));
        });
    }
    // Every ticket is worked on by all teams at once: team n % TEAMS steps its STEP part, the next team forms the psi of
    // its PSI part (with one team: both, one after the other)
    __device__ __forceinline__ void step_role(int team, unsigned n_mine, unsigned b0, unsigned stride) const {
        const int t = ((int)threadIdx.x - team * C::STEP_THREADS) * CPT;
        const int lane = (int)(threadIdx.x & 31), wid = (int)(threadIdx.x >> 5);
        unsigned cnt = 0;
        TileItem nxt = n_mine > 0 ? item_of(w.items, b0) : TileItem{0, 0, 0, 0, 0, 0, 0, 0};
        for (unsigned n = 0; n < n_mine; ++n) {
            const int stage = (int)(n % NS);
            const unsigned ph = (n / NS) & 1u;
            const TileItem it = nxt;                       // (loaded one ticket ahead)
            if (n + 1 < n_mine) nxt = item_of(w.items, b0 + (n + 1) * stride);
            const bool do_step = n % C::TEAMS == (unsigned)team;
            const bool do_psi = C::TEAMS == 1 || (n + 1) % C::TEAMS == (unsigned)team;
            // the team that steps waits for the STEP rows, the team that forms psi for the PSI rows; every step warp sees
            // every phase of both barriers before it lets go of the stage (a parity wait must never be asked about a phase
            // two ahead of the last one seen, and a stage is refilled only after all of its rows have landed)
            if (do_step && !mbar_wait(&full[2 * stage], ph, w.status, 1)) return;
            if (threadIdx.x == 0) TILE_TRACE(5, n);
#ifndef LBM_TILE_NOSTEP
            if (do_step && it.sv) {
                const TilePos sp{it.sx, it.sy, it.sz};
                if (t < min(TILE_TX, p.nx - sp.xs * TILE_TX)) {
                    if (edge_row(sp.y, sp.z)) step_cells<WALLYZ>(stage, sp, t); else step_cells<false>(stage, sp, t);
                }
            }
            if (!mbar_wait(&full[2 * stage + 1], ph, w.status, 1)) return;
            if (do_psi && it.pv) {
                const TilePos pp{it.px, it.py, it.pz};
                if (t < min(TILE_TX, p.nx - pp.xs * TILE_TX)) {
                    if (edge_row(pp.y, pp.z)) psi_cells<WALLYZ>(stage, pp, t); else psi_cells<false>(stage, pp, t);
                }
            }
#endif
            if (!do_step && !mbar_wait(&full[2 * stage], ph, w.status, 1)) return;
            __syncwarp();
            if (threadIdx.x == 0) TILE_TRACE(6, n);
            if (lane == 0) {
                // (the counter the publisher reads: STEP parts of this team's tickets, after the stores of the whole warp)
                if (do_step) st_release_cta_shared(&done[wid], ++cnt);
                mbar_arrive(&empty[stage]);
            }
        }
    }

    // ---------------- publisher ----------------
    // the flags of the tiles every step warp of this block has stored: one gpu-scope fence (cumulative over the
    // stores it has observed through the done counters), then the flags
    __device__ __forceinline__ void publish_role(unsigned n_mine, unsigned b0, unsigned stride) const {
        const int lane = (int)(threadIdx.x & 31);
        unsigned k[C::TEAMS], left = n_mine;
#pragma unroll
        for (int tm = 0; tm < C::TEAMS; ++tm) k[tm] = 0;
        long long t0 = clock64();
        while (left > 0) {
            bool any = false;
#pragma unroll
            for (int tm = 0; tm < C::TEAMS; ++tm) {
                unsigned m = ld_acquire_cta_shared(&done[tm * C::STEP_WARPS]);
#pragma unroll
                for (int q = 1; q < C::STEP_WARPS; ++q) m = min(m, ld_acquire_cta_shared(&done[tm * C::STEP_WARPS + q]));
                // one value for the whole warp: the lanes may have read the counters at different times (independent
                // thread scheduling), and each lane publishes the tickets k + lane, k + lane + 32, ... below m
                m = __shfl_sync(0xffffffffu, m, 0);
                if (m > k[tm]) {
                    fence_acq_rel_gpu();
                    for (unsigned j = k[tm] + lane; j < m; j += 32) {
                        const TileItem it = item_of(w.items, b0 + (j * C::TEAMS + tm) * stride);
                        if (it.sv) st_relaxed(flag_of(it.sx, it.sy, it.sz), w.epoch);
                    }
                    TILE_TRACE(2, (m - 1) * C::TEAMS + tm);
                    left -= m - k[tm];
                    k[tm] = m;
                    any = true;
                }
            }
            if (any) {
                t0 = clock64();
            } else {
                __nanosleep(200);
                if (clock64() - t0 > TILE_TIMEOUT_CYCLES) { atomicOr(w.status, 4); return; }
            }
        }
    }
};

template <class R, class L, int MODEL, int PARITY, bool WALLYZ, bool VSHIFT>
__global__ void __launch_bounds__(TileCfg<R, L, MODEL>::THREADS, 1)
k_tile(const __grid_constant__ KP<R> p, const __grid_constant__ TileArgs w) {
    using T = Tile<R, L, MODEL, PARITY, WALLYZ, VSHIFT>;
    using C = typename T::C;
    extern __shared__ __align__(128) unsigned char tile_smem[];
    const T tl(p, w, tile_smem);
    const int wid = (int)(threadIdx.x >> 5);
    if (threadIdx.x == 0) {
        for (int s = 0; s < C::NS; ++s) {
            mbar_init(&tl.full[2 * s], 33 * C::PROD_S);       // per producer warp: one expect_tx arrival, 32 cp.async arrivals
            mbar_init(&tl.full[2 * s + 1], 33 * C::PROD_P);
            mbar_init(&tl.empty[s], C::TEAMS * C::STEP_WARPS);
        }
        for (int k = 0; k < 8; ++k) tl.done[k] = 0u;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // static work distribution: block b owns the STEP tickets b, b + gridDim.x, ...
    const unsigned b0 = blockIdx.x, stride = gridDim.x;
    const unsigned n_mine = b0 < w.n_items ? (w.n_items - b0 + stride - 1) / stride : 0u;
    // warp roles: the step warps have the lowest warp ids, the (short, latency-critical) producers the highest -- the warp
    // scheduler favours the highest id among the eligible warps of a sub-partition
    constexpr int SW = C::TEAMS * C::STEP_WARPS;
    if (wid < SW) tl.step_role(wid / C::STEP_WARPS, n_mine, b0, stride);
    else if (wid == SW) tl.publish_role(n_mine, b0, stride);
    else if (wid <= SW + C::PROD_P) tl.template produce<1>(wid - (SW + 1), C::PROD_P, n_mine, b0, stride);
    else tl.template produce<0>(wid - (SW + 1 + C::PROD_P), C::PROD_S, n_mine, b0, stride);
}

}  // namespace lbm
