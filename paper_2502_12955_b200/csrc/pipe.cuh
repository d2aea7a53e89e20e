// Pipelined persistent step kernel (sm_100a): the populations (and, for Shan-Chen models, the psi tile with
// its one-cell halo) of a 128-cell x-row segment are staged in shared memory with 16-byte asynchronous copies
// (cp.async.cg -> LDGSTS.128), double buffered, so that the loads of the NEXT segment are in flight while the
// current one is collided.  Bytes in flight cost no registers, one copy instruction moves 16 bytes (4 / 2
// cells) instead of one load per cell and slot, the collide code reads shared memory at compile-time offsets,
// and the psi stencil (Eq. 11 / 13) takes its 18 (8 in 2D) neighbours from the tile.
//
// Shan-Chen models run the psi pass (a2) and the fused step (a1, a3-a8) of one time step in this ONE launch:
// psi^sigma(x + c_i, t) must be known for all neighbours before cell x is collided (R9), and with in-place
// streaming a cell's populations can only be read before its own step overwrites them, so a separate psi pass
// has to re-read every population from HBM.  Here a psi item reads the populations of a segment (first touch,
// from HBM) and publishes psi; the step item of the same segment follows a short distance later in the
// schedule (wave_schedule.h) and finds them in L2.
//
// Work distribution: a global ticket counter hands out the items of the schedule in order.  A psi item never
// waits.  A step item waits for the published psi of the (up to) 27 segments around it, all of which have
// LOWER tickets.  Thread 0 keeps two more tickets in flight (one whose item is being loaded, one whose atomic
// is pending), so neither latency sits on the critical path.  Blocks process their tickets in increasing
// order and only ever wait on lower tickets, so the lowest unfinished ticket is always some block's current
// item and can proceed: no deadlock for any number of resident blocks.  A wait that does not end within a
// bounded number of polls sets *status and gives up (the host reports it) instead of hanging the GPU.
//
// Publication: every thread stores its psi values; __syncthreads; thread 0 stores the launch epoch into the
// segment's flag with release semantics at gpu scope.  Consumption: lanes of warp 0 poll the flags with
// acquire loads; __syncthreads; the psi tile is then copied with cp.async.cg (L2, never a stale L1 line).
//
// Requirements (checked by the host, otherwise k_step / k_psi run): nx * sizeof(R) a multiple of 16 bytes
// (every row starts 16-byte aligned), periodic x (walls in y / z are uniform per row and handled here).
//
// In-place (AA) streaming as in kernels.cuh: row r of a stage holds, for the cells x0..x0+len-1 of the
// segment, the slot P_i(x) of one direction i; for odd parity that is slot opp(i) of the row (y - c_y, z - c_z)
// shifted by -c_x in x, so the copy brings the aligned segment plus the 16-byte piece left or right of it
// (periodic wrap) and thread t reads position H + t - c_x.  Pieces contain elements owned by other cells
// (possibly being rewritten by their owners): those are never used.
#pragma once
#include "kernels.cuh"
#include "wave_schedule.h"

namespace lbm {

constexpr int PIPE_TX = 128;    // cells per segment = threads per block
enum { ITEM_STEP = 0, ITEM_PSI = 1, ITEM_END = 2 };

// one schedule entry per ticket (host-built, wave_schedule.h): kind, x-segment, y, z
struct PipeItem {
    int kind, xs, y, z;
};

struct PipeArgs {
    const PipeItem* items;          // the schedule of one time step (device)
    unsigned n_tickets;
    int nxs;                        // x-segments of PIPE_TX cells per row
    int* flags;                     // one per segment (z, y, xs): epoch of the last published psi
    unsigned long long* counter;    // ticket counter, never reset between launches
    unsigned long long base;        // counter value at which this launch starts
    int epoch;                      // > 0, differs from every earlier launch since the flags were cleared
    int* status;                    // set to 1 if a wait timed out
};

__device__ __forceinline__ int ld_acquire(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void cp_async16(unsigned smem_dst, const void* gmem_src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_dst), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <class R>
struct PipeGeom {
    static constexpr int H = 16 / (int)sizeof(R);    // elements per 16-byte piece = halo width in elements
    static constexpr int RS = PIPE_TX + 2 * H;       // elements per shared-memory row: [halo | segment | halo]
    static constexpr int PPR = PIPE_TX / H;          // pieces per full segment: 32 (fp32), 64 (fp64)
};

// rows of one stage: S*Q flow rows, Qs scalar rows, then S*NPSI psi rows ((dy, dz) in {-1,0,1}^2, 2D: dy only)
template <class L, int MODEL>
struct PipeRows {
    using MT = ModelTraits<MODEL>;
    using LS = typename ScalarOf<L>::type;
    static constexpr int NF = MT::S * L::Q;
    static constexpr int NH = MT::SCALAR ? LS::Q : 0;
    static constexpr int NPOPS = NF + NH;
    static constexpr int NPSI = L::D == 3 ? 9 : 3;
    static constexpr int NP = MT::SC ? MT::S * NPSI : 0;
    static constexpr int NR = NPOPS + NP;
    __host__ __device__ static constexpr int psi_row(int s, int cy, int cz) {
        return NPOPS + s * NPSI + (cy + 1) + (L::D == 3 ? 3 * (cz + 1) : 0);
    }
};

// per row, independent of the item: where the row comes from relative to the item's (y, z)
struct RowConst {
    unsigned long long base;    // global address of element 0 of the slot array the row is taken from
    unsigned long long own;     // the same for "slot i of the cell itself" (used beyond a bounce-back wall)
    int dy, dz, sx, pad;
};

template <class R, class L, int MODEL>
constexpr size_t pipe_smem_bytes() {
    using G = PipeGeom<R>;
    using T = PipeRows<L, MODEL>;
    return 2 * (size_t)T::NR * G::RS * sizeof(R)                       // two stages of rows
           + 3 * (size_t)T::NR * (sizeof(unsigned long long) + sizeof(int))   // row tables of three items in flight
           + (size_t)T::NR * sizeof(RowConst) + 16;
}

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

// are the psi values of the (up to) 27 segments around (xs, m, s) published?  All 32 lanes of a warp call it.
// blocking: poll until they are (bounded; on timeout *status = 1 and the result is "ready").
__device__ __forceinline__ bool psi_published(const PipeArgs& w, int xs, int m, int s, int nm, int ns, bool blocking) {
    const int l = (int)(threadIdx.x & 31);
    bool ok = true;
    if (l < 27) {
        const int dx = l % 3 - 1, dm = (l / 3) % 3 - 1, ds = l / 9 - 1;
        int xx = xs + dx, mm = m + dm, ss = s + ds;
        xx = xx < 0 ? xx + w.nxs : (xx >= w.nxs ? xx - w.nxs : xx);
        mm = mm < 0 ? mm + nm : (mm >= nm ? mm - nm : mm);
        ss = ss < 0 ? ss + ns : (ss >= ns ? ss - ns : ss);
        const int* fl = w.flags + ((size_t)ss * nm + mm) * w.nxs + xx;
        ok = ld_acquire(fl) == w.epoch;
        if (blocking) {
            unsigned spins = 0;
            while (!ok) {
                __nanosleep(32);
                ok = ld_acquire(fl) == w.epoch;
                if (++spins > (1u << 24)) { *w.status = 1; ok = true; }
            }
        }
    }
    return __all_sync(0xffffffffu, ok);
}

template <class R, class L, int MODEL, int PARITY, bool WALLYZ, bool FORCED>
struct Pipe {
    using G = PipeGeom<R>;
    using T = PipeRows<L, MODEL>;
    using MT = ModelTraits<MODEL>;
    using LS = typename ScalarOf<L>::type;
    static constexpr int S = MT::S, Q = L::Q, D = L::D, H = G::H, RS = G::RS, PPR = G::PPR, NR = T::NR;
    static constexpr int B = (int)sizeof(R);
    static constexpr int NW = PIPE_TX / 32;

    // views of the dynamic shared memory
    R* rows;                        // [2][NR][RS]
    unsigned long long* rowptr;     // [3][NR]: global address of element x = 0 of the row staged in row r
    int* rowsx;                     // [3][NR]: x-shift of the row (-1, 0, +1): thread t reads position H + t + shift
    RowConst* rowconst;             // [NR]
    const KP<R>& p;

    __device__ __forceinline__ Pipe(const KP<R>& kp, unsigned char* smem) : p(kp) {
        rows = (R*)smem;
        rowptr = (unsigned long long*)(smem + 2 * (size_t)NR * RS * sizeof(R));
        rowsx = (int*)(rowptr + 3 * NR);
        rowconst = (RowConst*)(((size_t)(rowsx + 3 * NR) + 15) & ~(size_t)15);
    }
    static __device__ __forceinline__ int wrap(int v, int n) { return v < 0 ? v + n : (v >= n ? v - n : v); }

    // once per block: thread r fills rowconst[r]
    __device__ __forceinline__ void init_row_const(int r) const {
        const size_t N = (size_t)p.N;
        RowConst rc;
        rc.dy = rc.dz = rc.sx = rc.pad = 0;
        if (r < T::NPOPS) {
            int i, c0, c1, c2, op;
            const R* arr;
            if (r < T::NF) {
                const int s = r / Q;
                i = r - s * Q;
                arr = p.f + (size_t)s * Q * N;
                c0 = c_runtime<L, 0>(i); c1 = c_runtime<L, 1>(i); c2 = c_runtime<L, 2>(i); op = L::opp(i);
            } else {
                i = r - T::NF;
                arr = p.h;
                c0 = c_runtime<LS, 0>(i); c1 = c_runtime<LS, 1>(i); c2 = c_runtime<LS, 2>(i); op = LS::opp(i);
            }
            rc.own = (unsigned long long)(arr + (size_t)i * N);
            rc.base = rc.own;
            if (PARITY == 1 && i != 0) {
                // P_i(x) = slot opp(i) of cell x - c_i (or slot i of x itself beyond a bounce-back wall)
                rc.base = (unsigned long long)(arr + (size_t)op * N);
                rc.sx = -c0; rc.dy = -c1; rc.dz = -c2;
            }
        } else {
            const int q = r - T::NPOPS;
            const int s = q / T::NPSI, k = q - s * T::NPSI;
            rc.base = rc.own = (unsigned long long)(p.psi + (size_t)s * N);
            rc.dy = k % 3 - 1;
            rc.dz = D == 3 ? k / 3 - 1 : 0;
        }
        rowconst[r] = rc;
    }

    // which global row does stage row r hold for an item at (y, z)?
    __device__ __forceinline__ void setup_row(int tbl, int r, int y, int z) const {
        const RowConst rc = rowconst[r];
        int yy = y + rc.dy, zz = z + rc.dz, sx = rc.sx;
        unsigned long long b = rc.base;
        if (WALLYZ) {
            const bool cross = (p.bc[1] && (yy < 0 || yy >= p.ny)) || (D == 3 && p.bc[2] && (zz < 0 || zz >= p.nz));
            if (cross) { b = rc.own; yy = y; zz = z; sx = 0; }
        }
        yy = wrap(yy, p.ny);
        zz = D == 3 ? wrap(zz, p.nz) : 0;
        rowptr[tbl * NR + r] = b + (((size_t)zz * p.ny + yy) * (size_t)p.nx) * B;
        rowsx[tbl * NR + r] = sx;
    }
    __device__ __forceinline__ void setup_item(int tbl, const PipeItem& it) const {   // one warp
        const int nrows = it.kind == ITEM_PSI ? T::NF : NR;
        for (int r = (int)(threadIdx.x & 31); r < nrows; r += 32) setup_row(tbl, r, it.y, it.z);
    }

    // asynchronous copies of rows [R0, R1) of the segment starting at x0 (len cells): warp w takes rows
    // R0 + w, R0 + w + 4, ..., lane l the 16-byte piece l (and l + 32 for fp64); then one thread per row
    // fetches the halo piece(s): both for psi rows, else the side the row's x-shift points to
    template <int R0, int R1, bool BOTH>
    __device__ __forceinline__ void issue_rows(int stage, int tbl, int x0, int len) const {
        const int t = (int)threadIdx.x, wid = t >> 5, lane = t & 31;
        const int pieces = len / H;
        const unsigned sbase = (unsigned)__cvta_generic_to_shared(rows) +
                               (unsigned)((((stage * NR + wid) * RS) + H + lane * H) * B);
        const unsigned long long* tb = rowptr + tbl * NR + wid;
        const unsigned lb = (unsigned)((x0 + lane * H) * B);
        static_for<0, (R1 - R0 + NW - 1) / NW>([&](auto kc) {
            constexpr int k = decltype(kc)::value;
            constexpr int rr = R0 + k * NW;                  // + wid
            if (rr + NW <= R1 || rr + wid < R1) {
                const char* g = (const char*)tb[rr] + lb;
                if (lane < pieces) cp_async16(sbase + (unsigned)(rr * RS * B), g);
                if constexpr (PPR > 32) {
                    if (lane + 32 < pieces) cp_async16(sbase + (unsigned)(rr * RS * B + 32 * H * B), g + 32 * H * B);
                }
            }
        });
        if (t < R1 - R0) {
            const int r = R0 + t;
            const int sx = rowsx[tbl * NR + r];
            const char* g0 = (const char*)rowptr[tbl * NR + r];
            const unsigned d0 = (unsigned)__cvta_generic_to_shared(rows) + (unsigned)(((stage * NR + r) * RS) * B);
            if (BOTH || sx < 0) {
                const int xl = x0 == 0 ? p.nx - H : x0 - H;
                cp_async16(d0, g0 + (size_t)xl * B);
            }
            if (BOTH || sx > 0) {
                const int xr = x0 + len == p.nx ? 0 : x0 + len;
                cp_async16(d0 + (unsigned)((H + len) * B), g0 + (size_t)xr * B);
            }
        }
    }
    __device__ __forceinline__ void issue_pops(int stage, int tbl, const PipeItem& it) const {
        const int x0 = it.xs * PIPE_TX;
        const int len = min(PIPE_TX, p.nx - x0);
        if (it.kind == ITEM_PSI) issue_rows<0, T::NF, false>(stage, tbl, x0, len);
        else issue_rows<0, T::NPOPS, false>(stage, tbl, x0, len);
    }
    __device__ __forceinline__ void issue_psi(int stage, int tbl, const PipeItem& it) const {
        const int x0 = it.xs * PIPE_TX;
        const int len = min(PIPE_TX, p.nx - x0);
        if constexpr (T::NP > 0) issue_rows<T::NPOPS, NR, true>(stage, tbl, x0, len);
    }

    // x-shift of the row holding direction I of lattice LL: a compile-time constant unless the item touches
    // a bounce-back wall (EDGE), where rows may have been redirected to the cell's own slot
    template <class LL, int I, bool EDGE>
    __device__ __forceinline__ int shift_of(int tbl, int r) const {
        if constexpr (PARITY == 0 || I == 0) return 0;
        else if constexpr (EDGE) return rowsx[tbl * NR + r];
        else return -LL::c(I, 0);
    }
    // populations of lattice LL staged in rows R0.. -> registers; sb = this thread's position in row 0
    template <class LL, int R0, bool EDGE>
    __device__ __forceinline__ void read_pops(const R* sb, int tbl, R* fl) const {
        static_for<0, LL::Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            fl[i] = sb[(R0 + i) * RS + shift_of<LL, i, EDGE>(tbl, R0 + i)];
        });
    }
    // f*_{opp(i)} back to P_i(x): the global row the stage row came from, column x + shift (periodic wrap)
    template <class LL, int R0, bool EDGE>
    __device__ __forceinline__ void write_pops(int tbl, const unsigned* col, const R* fl) const {
        static_for<0, LL::Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            const int sx = shift_of<LL, i, EDGE>(tbl, R0 + i);
            R* g0 = (R*)rowptr[tbl * NR + R0 + i];
            g0[sx < 0 ? col[0] : (sx > 0 ? col[2] : col[1])] = fl[LL::opp(i)];
        });
    }

    // step a2 for the segment: rho^sigma in index order (Eq. 7 / 18), psi^sigma (Eq. 10 / 24 or psi = rho)
    __device__ __forceinline__ void compute_psi(int stage, int tbl, const PipeItem& it) const {
        const int t = (int)threadIdx.x, x = it.xs * PIPE_TX + t;
        if (x >= p.nx) return;
        const R* sb = rows + (size_t)stage * NR * RS + H + t;
        const size_t cell = ((size_t)it.z * p.ny + it.y) * (size_t)p.nx + (size_t)x;
        static_for<0, S>([&](auto sc) {
            constexpr int s = decltype(sc)::value;
            R fl[Q];
            read_pops<L, s * Q, false>(sb, tbl, fl);
            R rho, j[3];
            moments<L>(fl, rho, j);
            p.psi[(size_t)s * (size_t)p.N + cell] = psi_of(rho, p.psi_kind, p.rho0_psi);
        });
    }

    // steps a1, a3-a8 for the segment
    template <bool EDGE>
    __device__ __forceinline__ void compute_step(int stage, int tbl, const PipeItem& it) const {
        const int t = (int)threadIdx.x, x = it.xs * PIPE_TX + t;
        if (x >= p.nx) return;
        const R* sb = rows + (size_t)stage * NR * RS + H + t;
        R fl[S][Q];
        static_for<0, S>([&](auto sc) {
            constexpr int s = decltype(sc)::value;
            read_pops<L, s * Q, EDGE>(sb, tbl, fl[s]);
        });
        R hl[LS::Q];
        if constexpr (MT::SCALAR) read_pops<LS, T::NF, EDGE>(sb, tbl, hl);

        R acc[S][3], psi_own[S];
        if constexpr (MT::SC) {
            // stencil sums from the shared-memory psi tile, same order of additions as sc_stencil
            static_for<0, S>([&](auto tc) {
                constexpr int tt = decltype(tc)::value;
                acc[tt][0] = acc[tt][1] = acc[tt][2] = (R)0;
                static_for<1, Q>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    constexpr int CX = L::c(i, 0), CY = L::c(i, 1), CZ = L::c(i, 2);
                    const R pv = sb[T::psi_row(tt, CY, CZ) * RS + CX];
                    static_for<0, D>([&](auto ac) {
                        constexpr int a = decltype(ac)::value;
                        constexpr int c = L::c(i, a);
                        if constexpr (c != 0) acc[tt][a] = vfma((R)(c * L::w(i)), pv, acc[tt][a]);
                    });
                });
                psi_own[tt] = sb[T::psi_row(tt, 0, 0) * RS];
            });
        }
        CellMacro<R, L, MODEL> m;
        cell_macros_core<R, L, MODEL, FORCED>(p, fl, acc, psi_own, m);

        // columns x-1, x, x+1 (periodic wrap) within a global row
        unsigned col[3];
        col[0] = (unsigned)(x == 0 ? p.nx - 1 : x - 1);
        col[1] = (unsigned)x;
        col[2] = (unsigned)(x == p.nx - 1 ? 0 : x + 1);
        static_for<0, S>([&](auto sc) {
            constexpr int s = decltype(sc)::value;
            collide_component<R, L, FORCED, s>(p, fl[s], m.rho[s], m.u, m.F[s]);
            write_pops<L, s * Q, EDGE>(tbl, col, fl[s]);
        });
        if constexpr (MT::SCALAR) {
            collide_scalar<R, LS>(p, hl, m.rho[0], m.rho[S - 1], m.inv_rho, m.u);
            write_pops<LS, T::NF, EDGE>(tbl, col, hl);
        }
    }
};

template <class R, class L, int MODEL, int PARITY, bool WALLYZ, bool FORCED>
__global__ void __launch_bounds__(PIPE_TX) k_pipe(const __grid_constant__ KP<R> p, const __grid_constant__ PipeArgs w) {
    using P = Pipe<R, L, MODEL, PARITY, WALLYZ, FORCED>;
    using T = typename P::T;
    constexpr bool SC = ModelTraits<MODEL>::SC;
    constexpr int D = L::D;
    extern __shared__ __align__(16) unsigned char pipe_smem[];
    __shared__ PipeItem s_item[2];
    __shared__ int s_ready;
    const P pp(p, pipe_smem);
    const int t = (int)threadIdx.x, wid = t >> 5, lane = t & 31;
    const int nm = D == 3 ? p.ny : 1, ns = D == 3 ? p.nz : p.ny;

    // lane 0 of warp 0: ticket pipeline.  it1: item of the next-but-one ticket (loaded or loading);
    // tk2: the ticket after that (atomic pending)
    auto take = [&]() -> unsigned { return (unsigned)(atomicAdd(w.counter, 1ULL) - w.base); };
    auto load_item = [&](unsigned tk) -> PipeItem {
        PipeItem it{ITEM_END, 0, 0, 0};
        if (tk < w.n_tickets) {
            const int4 v = __ldg((const int4*)(w.items + tk));
            it.kind = v.x; it.xs = v.y; it.y = v.z; it.z = v.w;
        }
        return it;
    };
    auto bcast = [&](PipeItem it) -> PipeItem {
        it.kind = __shfl_sync(0xffffffffu, it.kind, 0);
        it.xs = __shfl_sync(0xffffffffu, it.xs, 0);
        it.y = __shfl_sync(0xffffffffu, it.y, 0);
        it.z = __shfl_sync(0xffffffffu, it.z, 0);
        return it;
    };
    auto m_of = [&](const PipeItem& it) { return D == 3 ? it.y : 0; };
    auto s_of = [&](const PipeItem& it) { return D == 3 ? it.z : it.y; };
    auto is_edge = [&](const PipeItem& it) {
        return WALLYZ && ((p.bc[1] && (it.y == 0 || it.y == p.ny - 1)) || (D == 3 && p.bc[2] && (it.z == 0 || it.z == p.nz - 1)));
    };

    if (t < T::NR) pp.init_row_const(t);
    __syncthreads();
    unsigned tk2 = 0;
    PipeItem it1{ITEM_END, 0, 0, 0};
    if (wid == 0) {
        PipeItem first{ITEM_END, 0, 0, 0};
        if (lane == 0) {
            const unsigned a = take();
            const unsigned b = take();
            tk2 = take();
            first = load_item(a);
            it1 = load_item(b);
        }
        first = bcast(first);
        if (lane == 0) s_item[0] = first;
        if (first.kind != ITEM_END) pp.setup_item(0, first);
    }
    __syncthreads();
    PipeItem cur = s_item[0];
    int stage = 0, tbl = 0;
    bool cur_psi = false;       // psi tile of the current item already requested
    if (cur.kind != ITEM_END) pp.issue_pops(0, 0, cur);
    cp_async_commit();
    for (int k = 0; cur.kind != ITEM_END; ++k) {
        const int tbl_n = tbl == 2 ? 0 : tbl + 1;
        const bool need_psi = SC && cur.kind == ITEM_STEP && !cur_psi;
        if (wid == 0) {
            // the next item: publish it, work out its rows, look whether its psi is there already
            PipeItem n = it1;
            if (lane == 0) {
                it1 = load_item(tk2);
                tk2 = take();
            }
            n = bcast(n);
            if (lane == 0) s_item[(k + 1) & 1] = n;
            if (n.kind != ITEM_END) pp.setup_item(tbl_n, n);
            if (SC) {
                if (n.kind == ITEM_STEP) {
                    const bool r = psi_published(w, n.xs, m_of(n), s_of(n), nm, ns, false);
                    if (lane == 0) s_ready = r ? 1 : 0;
                }
                if (need_psi) psi_published(w, cur.xs, m_of(cur), s_of(cur), nm, ns, true);
            }
        }
        __syncthreads();                               // next item visible; the other stage is free; psi published
        const PipeItem nxt = s_item[(k + 1) & 1];
        if (SC && need_psi) pp.issue_psi(stage, tbl, cur);
        cp_async_commit();                             // group A (may be empty)
        bool nxt_psi = false;
        if (nxt.kind != ITEM_END) {
            pp.issue_pops(stage ^ 1, tbl_n, nxt);
            if (SC && nxt.kind == ITEM_STEP && s_ready) { pp.issue_psi(stage ^ 1, tbl_n, nxt); nxt_psi = true; }
        }
        cp_async_commit();                             // group B: prefetch of the next item
        cp_async_wait<1>();                            // everything but group B has landed (this thread's copies)
        __syncthreads();                               // ... and everybody else's
        if (cur.kind == ITEM_PSI) {
            if constexpr (SC) {
                pp.compute_psi(stage, tbl, cur);
                __syncthreads();
                if (t == 0) st_release(w.flags + ((size_t)s_of(cur) * nm + m_of(cur)) * w.nxs + cur.xs, w.epoch);
            }
        } else {
            if (WALLYZ && is_edge(cur)) pp.template compute_step<WALLYZ>(stage, tbl, cur);
            else pp.template compute_step<false>(stage, tbl, cur);
        }
        cur = nxt;
        cur_psi = nxt_psi;
        stage ^= 1;
        tbl = tbl_n;
    }
    cp_async_wait<0>();
}

}  // namespace lbm
