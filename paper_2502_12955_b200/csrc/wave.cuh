// Wavefront kernel of the Shan-Chen models: the psi pass (a2) and the fused step (a1, a3-a8) of ONE time
// step in ONE persistent launch, so that the populations cross HBM once per step (the psi item of a row
// reads them from HBM, the step item of the same row, a short distance later in the schedule, from L2).
// Schedule and the rule it obeys: wave_schedule.h.
//
// Work distribution: a global ticket counter hands out (row item, x-segment) pairs in schedule order.  A psi
// item never waits.  A step item waits for the published psi of the (up to) 27 chunks around it; all of them
// have LOWER tickets (their row items come earlier in the list), and tickets are only taken by running
// blocks, so every wait is on a block that is already resident and never waits itself: no deadlock, whatever
// the number of resident blocks.  A wait that does not end within a bounded number of polls sets *status and
// gives up (the host reports it) instead of hanging the GPU.
//
// Publication: every thread stores its psi values; __syncthreads; thread 0 stores the launch epoch into the
// chunk's flag with release semantics at gpu scope.  Consumption: lanes of warp 0 poll the flags with acquire
// loads; __syncthreads; psi is then read with ld.global.cg (L2), never through a possibly stale L1 line.
#pragma once
#include "kernels.cuh"
#include "wave_schedule.h"

namespace lbm {

struct WaveArgs {
    const WaveItem* items;          // row items of one time step (device)
    long long n_tickets;            // items * nxs
    int nxs;                        // x-segments (chunks of WAVE_SEG cells) per row
    int* flags;                     // one per chunk (z, y, xs): epoch of the last published psi
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

constexpr int WAVE_SEG = 128;   // cells per x-segment = threads per block

template <class R, class L, int MODEL, int PARITY>
__global__ void __launch_bounds__(WAVE_SEG) k_wave(const __grid_constant__ KP<R> p, const __grid_constant__ WaveArgs w) {
    __shared__ long long s_ticket;
    constexpr int D = L::D;
    const int nm = D == 3 ? p.ny : 1, ns = D == 3 ? p.nz : p.ny;
    for (;;) {
        if (threadIdx.x == 0) s_ticket = (long long)(atomicAdd(w.counter, 1ULL) - w.base);
        __syncthreads();
        const long long tk = s_ticket;
        __syncthreads();
        if (tk >= w.n_tickets) break;
        const long long ri = tk / w.nxs;
        const int xs = (int)(tk - ri * w.nxs);
        const WaveItem it = w.items[ri];
        const bool is_psi = it.m < 0;
        const int m = it.m & 0x7fffffff, s = it.s;
        const int y = D == 3 ? m : s, z = D == 3 ? s : 0;
        const int x = xs * WAVE_SEG + (int)threadIdx.x;
        if (is_psi) {
            if (x < p.nx) psi_cell<R, L, MODEL, PARITY>(p, x, y, z);
            __syncthreads();
            if (threadIdx.x == 0) st_release(w.flags + ((size_t)s * nm + m) * w.nxs + xs, w.epoch);
        } else {
            if (threadIdx.x < 32) {
                // lane -> neighbour chunk (dx, dm, ds) in {-1,0,1}^3, periodic wrap; lanes 27..31 idle
                const int l = (int)threadIdx.x;
                bool ok = true;
                if (l < 27) {
                    const int dx = l % 3 - 1, dm = (l / 3) % 3 - 1, ds = l / 9 - 1;
                    int xx = xs + dx, mm = m + dm, ss = s + ds;
                    xx = xx < 0 ? xx + w.nxs : (xx >= w.nxs ? xx - w.nxs : xx);
                    mm = mm < 0 ? mm + nm : (mm >= nm ? mm - nm : mm);
                    ss = ss < 0 ? ss + ns : (ss >= ns ? ss - ns : ss);
                    const int* fl = w.flags + ((size_t)ss * nm + mm) * w.nxs + xx;
                    ok = ld_acquire(fl) == w.epoch;
                    unsigned spins = 0;
                    while (!ok) {
                        __nanosleep(64);
                        ok = ld_acquire(fl) == w.epoch;
                        if (++spins > (1u << 24)) { *w.status = 1; break; }
                    }
                }
                __syncwarp();
            }
            __syncthreads();
            if (x < p.nx) step_cell<R, L, MODEL, PARITY, false, true, true>(p, x, y, z);
        }
    }
}

}  // namespace lbm
