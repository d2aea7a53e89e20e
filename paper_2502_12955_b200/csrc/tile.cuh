// Resident-tile kernel of the Shan-Chen models (sm_100a): ONE persistent, warp-specialised launch per time step in
// which every population crosses HBM once in each direction and is read from L2 once.
//
// The problem: Eq. 11 / 13 need psi(x + c_i, t) of all neighbours before cell x
// is collided (R9), and with in-place streaming a cell's populations can only be read before its own step
// overwrites them.  Two launches (k_psi, k_step) read the flow populations twice from HBM.  Here a block keeps the
// populations of a tile of TILE_TX cells of one x-row in SHARED MEMORY between the two uses:
//
//   producer warp   bulk-copies (cp.async.bulk -> UBLKCP, completion on an mbarrier) the S*Q + Q_s slot rows P_i(x) of
//                   the tile into the next free stage of a ring of NS stages; at odd parity a row comes from the
//                   neighbour row (y - c_y, z - c_z) and is shifted by -c_x, so it is the aligned segment plus the
//                   16-byte piece left or right of it.  One lane issues a row: no registers, no per-cell instructions.
//   psi warp        step a2: rho^sigma in index order (Eq. 7 / 18) from the stage, psi^sigma (Eq. 10 / 24 or psi = rho)
//                   to global memory, then publishes the tile's flag (st.release.gpu, launch epoch).
//   halo warp       waits (ld.acquire.gpu) for the flags of the up to 27 tiles around the tile -- published by the
//                   blocks that own them -- and copies the psi rows with their one-cell halo from L2 (cp.async.cg, never a stale L1 line) into one of TILE_NHB
//                   shared-memory halo buffers, without waiting for the copies.
//   step warps      steps a1, a3-a8: populations from the stage, psi stencil from the halo buffer, collide, store to
//                   the global slots the rows came from; in fp32 every thread owns TWO cells and runs the packed
//                   f32x2 instantiation (V = F2) of the cell arithmetic.
//
// Work distribution is static: block b owns the tickets b, b + B, b + 2B, ... of the host-built schedule
// (tile_schedule.h; one ticket = one tile), so every warp knows its items without communication.  Deadlock freedom:
// producer and psi warp never wait for another block (only for free stages and landed copies), the step of the
// globally lowest unreleased ticket g needs psi of tickets <= g + LEAD only, and every block keeps NS stages, i.e.
// its next NS tickets, loaded: with LEAD <= (NS - 1) * B all those tickets are in a stage, their psi gets published,
// and ticket g proceeds.  The host checks that inequality (lbm_set_path) and launches at most as many blocks as
// are co-resident.  Every wait is bounded (clock64); a timeout sets *status and gives up instead of hanging the GPU.
//
// Requirements (else the two-launch path runs): periodic x, nx * sizeof(R) a multiple of 16 bytes, no solid mask,
// Guo forcing.  Walls in y / z are uniform per row and handled here: rows beyond a wall are redirected to the
// cell's own slot (halfway bounce-back) and left out of the psi stencil (Eq. 11-12), adhesion Eq. 14 included.
#pragma once
#include "kernels.cuh"
#include "tile_schedule.h"

namespace lbm {

constexpr int TILE_TX = 128;          // cells per tile
// how the producer warp moves a row: 16-byte cp.async (LDGSTS.128) per lane, or one cp.async.bulk (UBLKCP) per row.
// The bulk form is the measured-and-rejected alternative (the per-SM request rate of 512-byte bulk
// copies bounds the kernel at about 1 TB/s); build with -DLBM_TILE_BULK=1 to reproduce it.
#ifndef LBM_TILE_BULK
#define LBM_TILE_BULK 0
#endif
constexpr bool TILE_BULK = LBM_TILE_BULK != 0;
constexpr int TILE_AUX_WARPS = 3;     // producer, psi, halo
#ifndef LBM_TILE_NHB
#define LBM_TILE_NHB 3
#endif
constexpr int TILE_NHB = LBM_TILE_NHB;   // psi halo buffers per block (the halo warp runs that many tiles ahead of the step warps)

struct TileItem {
    int kind, xs, y, z;               // TILE_FULL / TILE_PSI_ONLY, x-segment, row
};

struct TileArgs {
    const TileItem* items;            // the schedule of one time step, one entry per ticket (device)
    unsigned n_items;
    int nxs;                          // tiles per row
    int* flags;                       // one per tile (z, y, xs): launch epoch of the last published psi
    int epoch;                        // > 0, differs from every earlier launch since the flags were cleared
    int* status;                      // set to 1 if a wait timed out
#ifdef LBM_TILE_TRACE
    long long* trace;
#endif
};

#ifdef LBM_TILE_TRACE
// developer trace: time stamps of block 0's roles per item (0 issue, 1 full seen by psi, 2 psi published, 3 flags ok,
// 4 halo issued, 5 step start, 6 step end, 7 empty seen by the producer)
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
__device__ __forceinline__ int ld_acquire(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ int ld_relaxed(const int* p) {
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ void st_release(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ int4 ld_cg16(const void* p) {
    int4 v;
    asm volatile("ld.global.cg.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
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
// bounded wait for the phase with the given parity; false (and *status = 1) on timeout
__device__ __forceinline__ bool mbar_wait(unsigned long long* bar, unsigned parity, int* status) {
    if (mbar_try_wait(bar, parity)) return true;
    const long long t0 = clock64();
    while (!mbar_try_wait(bar, parity)) {
        if (clock64() - t0 > TILE_TIMEOUT_CYCLES) { *status = 1; return false; }
    }
    return true;
}
// 16-byte asynchronous copy global -> shared (LDGSTS.128, L2 only) and its completion on an mbarrier: the barrier
// receives one arrival from the executing thread once all its earlier cp.async have landed (.noinc: the arrival is
// part of the barrier's initial count)
// (no "memory" clobber: ordinary loads of the row tables may be scheduled across the copies; ordering against the
// consumers comes from the mbarrier operations, which do clobber memory)
__device__ __forceinline__ void cp_async16(unsigned dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src));
}
__device__ __forceinline__ void cp_async_arrive(unsigned long long* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// global -> shared bulk copy (bytes a multiple of 16, both addresses 16-byte aligned), completion counted on bar
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
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
template <class LL>
__host__ __device__ constexpr int count_x_shifted() {
    int n = 0;
    for (int i = 0; i < LL::Q; ++i) n += LL::c(i, 0) != 0;
    return n;
}

template <class R, class L, int MODEL, int NS>
struct TileCfg {
    using MT = ModelTraits<MODEL>;
    using LS = typename ScalarOf<L>::type;
    static constexpr bool PACK = sizeof(R) == 4;                 // two fp32 cells per step thread, packed arithmetic
    using V = std::conditional_t<PACK, F2, R>;
    static constexpr int CPT = PACK ? 2 : 1;
    static constexpr int S = MT::S, Q = L::Q, D = L::D;
    static constexpr int B = (int)sizeof(R);
    static constexpr int H = 16 / B;                             // elements per 16-byte piece = halo width
    static constexpr int RS = TILE_TX + 2 * H;                   // elements per shared-memory row: [piece | segment | piece]
    static constexpr int NF = S * Q;
    static constexpr int NH = MT::SCALAR ? LS::Q : 0;
    static constexpr int NPOPS = NF + NH;
    static constexpr int NPSI = D == 3 ? 9 : 3;                  // psi rows (dy, dz) per component
    static constexpr int NP = S * NPSI;
    static constexpr int STEP_THREADS = TILE_TX / CPT;
    static constexpr int STEP_WARPS = STEP_THREADS / 32;
    static constexpr int THREADS = 32 * TILE_AUX_WARPS + STEP_THREADS;
    static constexpr size_t STAGE_BYTES = (size_t)NPOPS * RS * B;
    static constexpr size_t HALO_BYTES = (size_t)NP * RS * B;
    static constexpr size_t ROWPTR_BYTES = (size_t)NS * NPOPS * sizeof(unsigned long long);
    static constexpr size_t ROWSX_BYTES = ((size_t)NS * NPOPS * sizeof(int) + 15) / 16 * 16;
    static constexpr int NBAR = 3 * NS + 2 * TILE_NHB;
    static constexpr size_t SMEM = NS * STAGE_BYTES + TILE_NHB * HALO_BYTES + ROWPTR_BYTES + ROWSX_BYTES + NBAR * 8;
    __host__ __device__ static constexpr int psi_row(int t, int cy, int cz) { return t * NPSI + (cy + 1) + (D == 3 ? 3 * (cz + 1) : 0); }
};

template <class R, class L, int MODEL, int PARITY, bool WALLYZ, int NS>
struct Tile {
    using C = TileCfg<R, L, MODEL, NS>;
    using MT = typename C::MT;
    using LS = typename C::LS;
    using V = typename C::V;
    static constexpr int S = C::S, Q = C::Q, D = C::D, B = C::B, H = C::H, RS = C::RS, NF = C::NF, NPOPS = C::NPOPS, CPT = C::CPT;

    const KP<R>& p;
    const TileArgs& w;
    R* stages;                          // [NS][NPOPS][RS]
    R* halo;                            // [TILE_NHB][NP][RS]
    unsigned long long* rowptr;         // [NS][NPOPS]: global address of element x = 0 of the row staged there
    int* rowsx;                         // [NS][NPOPS]: its x-shift (-1, 0, +1): cell x reads position H + (x - x0) + shift
    unsigned long long *full, *psi_done, *empty, *halo_full, *halo_empty;

    __device__ __forceinline__ Tile(const KP<R>& kp, const TileArgs& wa, unsigned char* smem) : p(kp), w(wa) {
        stages = (R*)smem;
        halo = (R*)(smem + NS * C::STAGE_BYTES);
        rowptr = (unsigned long long*)(smem + NS * C::STAGE_BYTES + TILE_NHB * C::HALO_BYTES);
        rowsx = (int*)((unsigned char*)rowptr + C::ROWPTR_BYTES);
        full = (unsigned long long*)((unsigned char*)rowsx + C::ROWSX_BYTES);
        psi_done = full + NS;
        empty = psi_done + NS;
        halo_full = empty + NS;
        halo_empty = halo_full + TILE_NHB;
    }
    static __device__ __forceinline__ int wrap(int v, int n) { return v < 0 ? v + n : (v >= n ? v - n : v); }
    __device__ __forceinline__ bool wall_y() const { return WALLYZ && p.bc[1]; }
    __device__ __forceinline__ bool wall_z() const { return WALLYZ && D == 3 && p.bc[2]; }
    // does the row offset (dy, dz) from row (y, z) cross a bounce-back wall?
    __device__ __forceinline__ bool crosses(int y, int z, int dy, int dz) const {
        if constexpr (!WALLYZ) return false;
        return (wall_y() && (y + dy < 0 || y + dy >= p.ny)) || (wall_z() && (z + dz < 0 || z + dz >= p.nz));
    }
    __device__ __forceinline__ TileItem item_of(unsigned ticket) const {
        const int4 v = __ldg((const int4*)(w.items + ticket));
        return TileItem{v.x, v.y, v.z, v.w};
    }

    // ---------------- producer ----------------
    // row r of a stage for an item at (y, z): slot array, source row, x-shift
    __device__ __forceinline__ void row_source(int r, int y, int z, unsigned long long& base, int& sx) const {
        const size_t N = (size_t)p.N;
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
        int slot = i, yy = y, zz = z;
        sx = 0;
        if (PARITY == 1 && i != 0 && !crosses(y, z, -c1, -c2)) {
            // P_i(x) = slot opp(i) of cell x - c_i; beyond a bounce-back wall: slot i of x itself
            slot = op; yy = wrap(y - c1, p.ny); zz = D == 3 ? wrap(z - c2, p.nz) : 0; sx = -c0;
        }
        base = (unsigned long long)(arr + (size_t)slot * N + ((size_t)zz * p.ny + yy) * (size_t)p.nx);
    }
    __device__ __forceinline__ void produce(unsigned n_mine, unsigned b0, unsigned stride) const {
        const int lane = (int)(threadIdx.x & 31);
        for (unsigned n = 0; n < n_mine; ++n) {
            const int stage = (int)(n % NS);
            const unsigned ph = (n / NS) & 1u;
            const TileItem it = item_of(b0 + n * stride);
            if (!mbar_wait(&empty[stage], ph ^ 1u, w.status)) return;
            TILE_TRACE(7, n);
            const int x0 = it.xs * TILE_TX;
            const int len = min(TILE_TX, p.nx - x0);
            const int nrows = it.kind == TILE_PSI_ONLY ? NF : NPOPS;
            // bytes this stage will receive: nrows segments plus one 16-byte piece per x-shifted row
            unsigned long long base[2] = {0, 0};
            int sx[2] = {0, 0};
            unsigned pieces = 0;
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const int r = lane + 32 * k;
                if (r < nrows) {
                    row_source(r, it.y, it.z, base[k], sx[k]);
                    rowptr[stage * NPOPS + r] = base[k];
                    rowsx[stage * NPOPS + r] = sx[k];
                    pieces += sx[k] != 0;
                }
            }
            pieces = __reduce_add_sync(0xffffffffu, pieces);
            __syncwarp();                                  // the row tables of all lanes are written
            TILE_TRACE(9, n);
            if constexpr (TILE_BULK) {
                // one cp.async.bulk (UBLKCP) per row and piece, completion as transaction bytes on the barrier
                if (lane == 0) mbar_arrive_expect_tx(&full[stage], (unsigned)nrows * (unsigned)(len * B) + 16u * pieces);
                __syncwarp();
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    const int r = lane + 32 * k;
                    if (r < nrows) {
                        const unsigned dst = smem_u32(stages + ((size_t)stage * NPOPS + r) * RS);
                        const char* g = (const char*)base[k];
                        bulk_g2s(dst + H * B, g + (size_t)x0 * B, (unsigned)(len * B), &full[stage]);
                        if (sx[k] < 0) bulk_g2s(dst, g + (size_t)(x0 == 0 ? p.nx - H : x0 - H) * B, 16u, &full[stage]);
                        if (sx[k] > 0) bulk_g2s(dst + (H + len) * B, g + (size_t)(x0 + len == p.nx ? 0 : x0 + len) * B, 16u, &full[stage]);
                    }
                }
            } else {
                // 16-byte cp.async (LDGSTS.128): lane l copies chunk l (and l + 32, ...) of every row, then the piece(s) of
                // its own rows; the barrier completes when the copies of all 32 lanes have landed
                const unsigned s0 = smem_u32(stages + (size_t)stage * NPOPS * RS) + (unsigned)((H + lane * H) * B);
                const unsigned goff = (unsigned)((x0 + lane * H) * B);
                const int nchunk = len / H;
                for (int r0 = 0; r0 < nrows; r0 += 8) {       // batches: 8 table reads, then 8 copies per lane
                    const char* g[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j) g[j] = (const char*)rowptr[stage * NPOPS + min(r0 + j, nrows - 1)] + goff;
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        if (r0 + j < nrows) {
                            const unsigned d = s0 + (unsigned)((r0 + j) * RS * B);
#pragma unroll
                            for (int q = 0; q < TILE_TX / H / 32; ++q)
                                if (lane + 32 * q < nchunk) cp_async16(d + (unsigned)(32 * q * H * B), g[j] + 32 * q * H * B);
                        }
                    }
                }
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    const int r = lane + 32 * k;
                    if (r < nrows && sx[k] != 0) {
                        const unsigned dst = smem_u32(stages + ((size_t)stage * NPOPS + r) * RS);
                        const char* g = (const char*)base[k];
                        if (sx[k] < 0) cp_async16(dst, g + (size_t)(x0 == 0 ? p.nx - H : x0 - H) * B);
                        else cp_async16(dst + (unsigned)((H + len) * B), g + (size_t)(x0 + len == p.nx ? 0 : x0 + len) * B);
                    }
                }
                cp_async_arrive(&full[stage]);
            }
            TILE_TRACE(0, n);
        }
    }

    // ---------------- reading a stage ----------------
    // population I of lattice LL (rows R0 ...) of the thread's cell(s); sb: position of the first cell in row 0 of the stage.
    // EDGE: the item touches a bounce-back wall, rows may have been redirected (shift from the table)
    template <class LL, int R0, int I, bool EDGE>
    __device__ __forceinline__ V read_pop(const R* sb, int stage) const {
        const R* q = sb + (R0 + I) * RS;
        if constexpr (PARITY == 0 || I == 0 || LL::c(I, 0) == 0) {
            if constexpr (C::PACK) { F2 v; v.v = *reinterpret_cast<const unsigned long long*>(q); return v; }
            else return *q;
        } else {
            int sh = -LL::c(I, 0);
            if constexpr (EDGE) sh = rowsx[stage * NPOPS + R0 + I];
            if constexpr (C::PACK) return pack2(q[sh], q[sh + 1]);
            else return q[sh];
        }
    }
    template <class LL, int R0, bool EDGE>
    __device__ __forceinline__ void read_pops(const R* sb, int stage, V* fl) const {
        static_for<0, LL::Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            fl[i] = read_pop<LL, R0, i, EDGE>(sb, stage);
        });
    }

    // ---------------- psi warp ----------------
    __device__ __forceinline__ void psi_role(unsigned n_mine, unsigned b0, unsigned stride) const {
        const int lane = (int)(threadIdx.x & 31);
        const int nm = D == 3 ? p.ny : 1;
        for (unsigned n = 0; n < n_mine; ++n) {
            const int stage = (int)(n % NS);
            const unsigned ph = (n / NS) & 1u;
            const TileItem it = item_of(b0 + n * stride);
            if (!mbar_wait(&full[stage], ph, w.status)) return;
            TILE_TRACE(1, n);
            const int x0 = it.xs * TILE_TX;
            const int len = min(TILE_TX, p.nx - x0);
            const bool edge = WALLYZ && ((wall_y() && (it.y == 0 || it.y == p.ny - 1)) || (wall_z() && (it.z == 0 || it.z == p.nz - 1)));
            const size_t row0 = ((size_t)it.z * p.ny + it.y) * (size_t)p.nx;
            // every lane takes its cell(s) of each 32 * CPT-cell chunk of the tile; the chunks are independent and
            // unrolled together, so that their (serial, index-ordered) sums overlap
            constexpr int NCH = TILE_TX / (32 * CPT);
            V ps[NCH][S];
#pragma unroll
            for (int c = 0; c < NCH; ++c) {
                const int t = c * 32 * CPT + lane * CPT;
                if (t < len) {
                    const R* sb = stages + (size_t)stage * NPOPS * RS + H + t;
                    static_for<0, S>([&](auto sc) {
                        constexpr int s = decltype(sc)::value;
                        V fl[Q];
                        if (WALLYZ && edge) read_pops<L, s * Q, true>(sb, stage, fl);
                        else read_pops<L, s * Q, false>(sb, stage, fl);
                        V rho = fl[0];
                        static_for<1, Q>([&](auto ic) { rho = rho + fl[decltype(ic)::value]; });      // Eq. 7 / 18, index order
                        ps[c][s] = psi_of(rho, p.psi_kind, p.rho0_psi);
                    });
                }
            }
#pragma unroll
            for (int c = 0; c < NCH; ++c) {
                const int t = c * 32 * CPT + lane * CPT;
                if (t < len) {
                    static_for<0, S>([&](auto sc) {
                        constexpr int s = decltype(sc)::value;
                        R* dst = p.psi + (size_t)s * (size_t)p.N + row0 + (size_t)(x0 + t);
                        if constexpr (C::PACK) *reinterpret_cast<unsigned long long*>(dst) = ps[c][s].v;
                        else *dst = ps[c][s];
                    });
                }
            }
            __syncwarp();
            if (lane == 0) {
                const int ms = D == 3 ? it.y : 0, ss = D == 3 ? it.z : it.y;
                st_release(w.flags + ((size_t)ss * nm + ms) * w.nxs + it.xs, w.epoch);
                mbar_arrive(&psi_done[stage]);
            }
            TILE_TRACE(2, n);
        }
    }

    // ---------------- halo warp ----------------
    // wait until the psi of the (up to) 27 tiles around (xs, y, z) is published
    __device__ __forceinline__ bool wait_flags(const TileItem& it) const {
        const int l = (int)(threadIdx.x & 31);
        const int nm = D == 3 ? p.ny : 1, ns = D == 3 ? p.nz : p.ny;
        const int m = D == 3 ? it.y : 0, s = D == 3 ? it.z : it.y;
        const bool wm = D == 3 ? wall_y() : false, wsl = D == 3 ? wall_z() : wall_y();
        bool ok = true;
        if (l < 27) {
            const int dx = l % 3 - 1, dm = (l / 3) % 3 - 1, ds = l / 9 - 1;
            int mm = m + dm, ss = s + ds;
            const bool beyond = (wm && (mm < 0 || mm >= nm)) || (wsl && (ss < 0 || ss >= ns)) || (D == 2 && dm != 0);
            if (!beyond) {
                const int xx = wrap(it.xs + dx, w.nxs);
                mm = wrap(mm, nm); ss = wrap(ss, ns);
                const int* fl = w.flags + ((size_t)ss * nm + mm) * w.nxs + xx;
                // relaxed polls (no L1 invalidation per poll), one acquire fence once every flag has been seen
                ok = ld_relaxed(fl) == w.epoch;
                if (!ok) {
                    const long long t0 = clock64();
                    while (!(ok = (ld_relaxed(fl) == w.epoch))) {
                        __nanosleep(100);
                        if (clock64() - t0 > TILE_TIMEOUT_CYCLES) { *w.status = 1; break; }
                    }
                }
            }
        }
        ok = __all_sync(0xffffffffu, ok);
        fence_acq_rel_gpu();                               // with the relaxed loads above: acquire of every flag
        __syncwarp();                                      // every lane's copies below come after every lane's acquire
        return ok;
    }
    __device__ __forceinline__ void halo_role(unsigned n_mine, unsigned b0, unsigned stride) const {
        const int lane = (int)(threadIdx.x & 31);
        unsigned h = 0;
        for (unsigned n = 0; n < n_mine; ++n) {
            const TileItem it = item_of(b0 + n * stride);
            if (it.kind != TILE_FULL) continue;
#ifndef LBM_TILE_NOWAIT
            if (!wait_flags(it)) return;
#endif
            TILE_TRACE(3, n);
            const int buf = (int)(h % TILE_NHB);
            if (!mbar_wait(&halo_empty[buf], ((h / TILE_NHB) & 1u) ^ 1u, w.status)) return;
            TILE_TRACE(8, n);
            const int x0 = it.xs * TILE_TX;
            const int len = min(TILE_TX, p.nx - x0);
            const int chunks = len / H + 2;                // segment plus one piece on either side
            const unsigned hb = smem_u32(halo + (size_t)buf * C::NP * RS);
            // asynchronous 16-byte copies (L2 only: cp.async.cg never reads a stale L1 line); the warp does not wait
            // for them but goes on to the flags of its next tile.  Per psi row: the segment chunks by all lanes,
            // the two 16-byte pieces left and right of it (periodic wrap in x) by lanes 0 and 1
            const int nchunk = len / H;
            const int xl = x0 == 0 ? p.nx - H : x0 - H, xr = x0 + len == p.nx ? 0 : x0 + len;
            // lane r < NP works out the source of psi row r (nullptr: beyond a wall, never read) ...
            const R* mine = nullptr;
            if (lane < C::NP) {
                const int t = lane / C::NPSI, q = lane - t * C::NPSI;
                const int dy = q % 3 - 1, dz = D == 3 ? q / 3 - 1 : 0;
                if (!crosses(it.y, it.z, dy, dz)) {
                    const int yy = wrap(it.y + dy, p.ny), zz = D == 3 ? wrap(it.z + dz, p.nz) : 0;
                    mine = p.psi + (size_t)t * (size_t)p.N + ((size_t)zz * p.ny + yy) * (size_t)p.nx;
                }
                // ... and copies its two pieces
                if (mine) {
                    const unsigned dst = hb + (unsigned)(lane * RS * B);
                    cp_async16(dst, mine + xl);
                    cp_async16(dst + (unsigned)((H + len) * B), mine + xr);
                }
            }
            // the segment of every row: chunk `lane` (and lane + 32, ...) by all lanes
#pragma unroll
            for (int row = 0; row < C::NP; ++row) {
                const R* src = (const R*)__shfl_sync(0xffffffffu, (unsigned long long)mine, row);
                if (src) {
                    const unsigned dst = hb + (unsigned)((row * RS + H) * B);
#pragma unroll
                    for (int k = 0; k < TILE_TX / H / 32; ++k)
                        if (lane + 32 * k < nchunk) cp_async16(dst + (unsigned)((lane + 32 * k) * H * B), src + x0 + (lane + 32 * k) * H);
                }
            }
            cp_async_arrive(&halo_full[buf]);
            TILE_TRACE(4, n);
            ++h;
        }
    }

    // ---------------- step warps ----------------
    // f*_{opp(i)} back to P_i(x): the global row the stage row came from, column x + shift (periodic wrap).
    // col[0..3] = x - 1, x, x + 1, x + 2 with wrap (x + 1 only for the second cell of a packed pair)
    template <class LL, int R0, int I, bool EDGE>
    __device__ __forceinline__ void write_pop(int stage, const int* col, V val) const {
        R* g0 = (R*)rowptr[stage * NPOPS + R0 + I];
        if constexpr (PARITY == 0 || I == 0 || LL::c(I, 0) == 0) {
            st_global(g0 + col[1], val);
        } else {
            int sh = -LL::c(I, 0);
            if constexpr (EDGE) sh = rowsx[stage * NPOPS + R0 + I];
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
    // psi of the thread's cell(s) at offset (CX, CY, CZ) from the halo buffer; hb: position of the first cell in row 0
    template <int CX, int CY, int CZ>
    __device__ __forceinline__ V psi_at(const R* hb, int t) const {
        const R* q = hb + C::psi_row(t, CY, CZ) * RS + CX;
        if constexpr (C::PACK) {
            if constexpr (CX == 0) { F2 v; v.v = *reinterpret_cast<const unsigned long long*>(q); return v; }
            else return pack2(q[0], q[1]);
        } else {
            return *q;
        }
    }
    template <bool EDGE>
    __device__ __forceinline__ void step_cells(int stage, int buf, const TileItem& it, int t) const {
        const int x = it.xs * TILE_TX + t;
        const R* sb = stages + (size_t)stage * NPOPS * RS + H + t;
        const R* hb = halo + (size_t)buf * C::NP * RS + H + t;
        V fl[S][Q];
        static_for<0, S>([&](auto sc) {
            constexpr int s = decltype(sc)::value;
            read_pops<L, s * Q, EDGE>(sb, stage, fl[s]);
        });
        V hl[LS::Q];
        if constexpr (MT::SCALAR) read_pops<LS, NF, EDGE>(sb, stage, hl);

        // stencil sums from the halo buffer, the order of sc_stencil (row a3)
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
                if (!out) pv = psi_at<CX, CY, CZ>(hb, tt);
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
            psi_own[tt] = psi_at<0, 0, 0>(hb, tt);
        });
        CellMacro<V, L, MODEL> m;
        cell_macros_core<V, L, MODEL, true, WALLYZ>(p, fl, acc, psi_own, m, adh);
        const int col[4] = {x == 0 ? p.nx - 1 : x - 1, x, x + 1 == p.nx ? 0 : x + 1, x + 2 >= p.nx ? x + 2 - p.nx : x + 2};
        static_for<0, S>([&](auto sc) {
            constexpr int s = decltype(sc)::value;
            collide_component<V, L, true, s>(p, fl[s], m.rho[s], m.u, m.F[s]);
            write_pops<L, s * Q, EDGE>(stage, col, fl[s]);
        });
        if constexpr (MT::SCALAR) {
            collide_scalar<V, LS>(p, hl, m.rho[0], m.rho[S - 1], m.inv_rho, m.u);
            write_pops<LS, NF, EDGE>(stage, col, hl);
        }
    }
    __device__ __forceinline__ void step_role(unsigned n_mine, unsigned b0, unsigned stride) const {
        const int t = (int)threadIdx.x * CPT;
        const int lane = (int)(threadIdx.x & 31);
        unsigned h = 0;
        for (unsigned n = 0; n < n_mine; ++n) {
            const int stage = (int)(n % NS);
            const unsigned ph = (n / NS) & 1u;
            const TileItem it = item_of(b0 + n * stride);
            if (!mbar_wait(&full[stage], ph, w.status)) return;
            if (!mbar_wait(&psi_done[stage], ph, w.status)) return;
            if (it.kind == TILE_FULL) {
                const int buf = (int)(h % TILE_NHB);
                if (!mbar_wait(&halo_full[buf], (h / TILE_NHB) & 1u, w.status)) return;
                if (threadIdx.x == 0) TILE_TRACE(5, n);
                const int len = min(TILE_TX, p.nx - it.xs * TILE_TX);
                if (t < len) {
                    const bool edge = WALLYZ && ((wall_y() && (it.y == 0 || it.y == p.ny - 1)) ||
                                                 (wall_z() && (it.z == 0 || it.z == p.nz - 1)));
                    if (WALLYZ && edge) step_cells<WALLYZ>(stage, buf, it, t);
                    else step_cells<false>(stage, buf, it, t);
                }
                __syncwarp();
                if (threadIdx.x == 0) TILE_TRACE(6, n);
                if (lane == 0) mbar_arrive(&halo_empty[buf]);
                ++h;
            } else {
                __syncwarp();
            }
            if (lane == 0) mbar_arrive(&empty[stage]);
        }
    }
};

template <class R, class L, int MODEL, int PARITY, bool WALLYZ, int NS>
__global__ void __launch_bounds__(TileCfg<R, L, MODEL, NS>::THREADS) k_tile(const __grid_constant__ KP<R> p, const __grid_constant__ TileArgs w) {
    using T = Tile<R, L, MODEL, PARITY, WALLYZ, NS>;
    using C = typename T::C;
    extern __shared__ __align__(128) unsigned char tile_smem[];
    const T tl(p, w, tile_smem);
    const int wid = (int)(threadIdx.x >> 5);
    if (threadIdx.x == 0) {
        for (int s = 0; s < NS; ++s) {
            mbar_init(&tl.full[s], TILE_BULK ? 1 : 32);
            mbar_init(&tl.psi_done[s], 1);
            mbar_init(&tl.empty[s], C::STEP_WARPS);
        }
        for (int b = 0; b < TILE_NHB; ++b) {
            mbar_init(&tl.halo_full[b], 32);
            mbar_init(&tl.halo_empty[b], C::STEP_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // static work distribution: block b owns the tickets b, b + gridDim.x, ...
    const unsigned b0 = blockIdx.x, stride = gridDim.x;
    const unsigned n_mine = b0 < w.n_items ? (w.n_items - b0 + stride - 1) / stride : 0u;
    // warp roles: the step warps have the lowest warp ids, the (short, latency-critical) producer the highest -- the warp
    // scheduler favours the highest id among the eligible warps of a sub-partition
    if (wid < C::STEP_WARPS) tl.step_role(n_mine, b0, stride);
    else if (wid == C::STEP_WARPS) tl.halo_role(n_mine, b0, stride);
    else if (wid == C::STEP_WARPS + 1) tl.psi_role(n_mine, b0, stride);
    else tl.produce(n_mine, b0, stride);
}

}  // namespace lbm
