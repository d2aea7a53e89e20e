// Wavefront kernel of the Shan-Chen models (register flavour): the psi segments (a2) and the step segments
// (a1, a3-a8) of ONE time step in ONE persistent launch, in the order of the host schedule (wave_schedule.h;
// ticket counter, flags and the deadlock argument as in pipe.cuh), but with the populations loaded straight
// into registers as in k_step.  A psi item reads a segment's populations from HBM and publishes psi; the step
// item of the same segment follows a short distance later and finds them in L2, so the populations cross HBM
// once per step.  Per item, lane 0 of warp 0 has the ticket, the schedule entry and the "psi is published"
// answer ready from the previous iteration; the population loads are issued BEFORE the block waits for the
// flags, so the wait costs nothing unless psi really is late.  psi is read with ld.global.cg (L2).
#pragma once
#include "pipe.cuh"

namespace lbm {

template <class R, class L, int MODEL, int PARITY>
__global__ void __launch_bounds__(PIPE_TX, StepBounds<R, MODEL, L::Q>::MINB) k_wave(const __grid_constant__ KP<R> p,
                                                                         const __grid_constant__ PipeArgs w) {
    using LS = typename ScalarOf<L>::type;
    constexpr int D = L::D, S = ModelTraits<MODEL>::S;
    __shared__ PipeItem s_item[2];
    __shared__ int s_ready[2];
    const int t = (int)threadIdx.x, wid = t >> 5, lane = t & 31;
    const int nm = D == 3 ? p.ny : 1, ns = D == 3 ? p.nz : p.ny;
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
        bool r = true;
        if (first.kind == ITEM_STEP) r = psi_published(w, first.xs, m_of(first), s_of(first), nm, ns, false);
        if (lane == 0) { s_item[0] = first; s_ready[0] = r ? 1 : 0; }
    }
    __syncthreads();
    PipeItem cur = s_item[0];
    bool ready = s_ready[0] != 0;
    for (int k = 0; cur.kind != ITEM_END; ++k) {
        const int x = cur.xs * PIPE_TX + t;
        const bool active = x < p.nx;
        const Nbr<D, false> nb(p, active ? x : 0, cur.y, cur.z);
        R fl[S][L::Q];
        R hl[LS::Q];
        // the populations first: they do not depend on psi
        if (active) {
            if (cur.kind == ITEM_STEP) step_load<R, L, MODEL, PARITY, false>(p, nb, fl, hl);
            else static_for<0, S>([&](auto sc) {
                constexpr int s = decltype(sc)::value;
                load_pops<L, PARITY, false>(p.f + (size_t)s * L::Q * (size_t)p.N, nb, (size_t)p.N, fl[s]);
            });
        }
        if (wid == 0) {
            PipeItem n = it1;
            if (lane == 0) {
                it1 = load_item(tk2);
                tk2 = take();
            }
            n = bcast(n);
            bool r = true;
            if (n.kind == ITEM_STEP) r = psi_published(w, n.xs, m_of(n), s_of(n), nm, ns, false);
            if (lane == 0) { s_item[(k + 1) & 1] = n; s_ready[(k + 1) & 1] = r ? 1 : 0; }
            if (cur.kind == ITEM_STEP && !ready) psi_published(w, cur.xs, m_of(cur), s_of(cur), nm, ns, true);
        }
        __syncthreads();
        if (cur.kind == ITEM_STEP) {
            if (active) step_finish<R, L, MODEL, PARITY, false, true, true>(p, nb, fl, hl);
        } else {
            if (active) {
                static_for<0, S>([&](auto sc) {
                    constexpr int s = decltype(sc)::value;
                    R rho, j[3];
                    moments<L>(fl[s], rho, j);
                    p.psi[(size_t)s * (size_t)p.N + nb.cell] = psi_of(rho, p.psi_kind, p.rho0_psi);
                });
            }
            __syncthreads();
            if (t == 0) st_release(w.flags + ((size_t)s_of(cur) * nm + m_of(cur)) * w.nxs + cur.xs, w.epoch);
        }
        cur = s_item[(k + 1) & 1];
        ready = s_ready[(k + 1) & 1] != 0;
    }
}

}  // namespace lbm
