// Launchers: runtime (model, parity, walls, forced) -> kernel template instance.
#pragma once
#include "dispatch.h"
#include "kernels.cuh"
#include "tile.cuh"
#include <cstdlib>

namespace lbm {

// threads per block: 128 (64 and 256 measured within 1 % for BGK, 256 slower for Shan-Chen), less for short rows
template <class R>
inline int block_for(const KP<R>& p) {
    int b = 128;
#ifdef LBM_TUNING
    if (const char* e = getenv("LBM_BLOCK")) b = atoi(e);
#endif
    while (b > 32 && b / 2 >= p.nx) b /= 2;
    return b;
}
// one block per segment of one x-row: grid (ceil(nx/block), ny, nz)
template <class R>
inline dim3 grid_for(const KP<R>& p) { const int b = block_for(p); return dim3((unsigned)((p.nx + b - 1) / b), (unsigned)p.ny, (unsigned)p.nz); }

template <class R, class L>
struct Launch {
    // run f(std::integral_constant<int, v>) for the run-time v in {0, ..., N-1}
    template <int N, class F>
    static bool with_int(int v, F&& f) {
        bool hit = false;
        static_for<0, N>([&](auto c) { if (decltype(c)::value == v) { f(c); hit = true; } });
        return hit;
    }
    template <class F>
    static bool with_sc_model(int model, F&& f) {
        switch (model) {
        case M_SC1: f(std::integral_constant<int, M_SC1>{}); return true;
        case M_SC2: f(std::integral_constant<int, M_SC2>{}); return true;
        case M_SC2_ADE: f(std::integral_constant<int, M_SC2_ADE>{}); return true;
        default: return false;
        }
    }

    // wmode: 0 fully periodic, 1 bounce-back walls (bc), 2 walls and / or a solid-node mask
    static cudaError_t psi(const void* kp, int model, int parity, int wmode, cudaStream_t st) {
        const KP<R>& p = *(const KP<R>*)kp;
        const bool ok = with_sc_model(model, [&](auto M) {
            with_int<3>(wmode, [&](auto W) {
                with_int<2>(parity, [&](auto P) {
                    k_psi<R, L, decltype(M)::value, decltype(P)::value, decltype(W)::value><<<grid_for(p), block_for(p), 0, st>>>(p);
                });
            });
        });
        return ok ? cudaGetLastError() : cudaErrorInvalidValue;
    }

    template <int MODEL, int WALLS, bool FORCED, bool VSHIFT = false, bool MOVING = false>
    static void step3(const KP<R>& p, int parity, cudaStream_t st) {
        if (parity) k_step<R, L, MODEL, 1, WALLS, FORCED, VSHIFT, MOVING><<<grid_for(p), block_for(p), 0, st>>>(p);
        else k_step<R, L, MODEL, 0, WALLS, FORCED, VSHIFT, MOVING><<<grid_for(p), block_for(p), 0, st>>>(p);
    }
    // forced: 0 no force, 1 Guo forcing (Eq. 20-23), 2 Shan-Chen velocity-shift forcing (Eq. 16-19);
    // moving: some wall has a velocity (Guo forcing only)
    static cudaError_t step(const void* kp, int model, int parity, int wmode, int forced, int moving, cudaStream_t st) {
        const KP<R>& p = *(const KP<R>*)kp;
        bool ok = false;
        if (moving) {
            if (forced == 2 || wmode == 0) return cudaErrorInvalidValue;
            ok = with_int<3>(wmode, [&](auto W) {
                constexpr int w = decltype(W)::value;
                if constexpr (w != 0) {
                    if (model == M_BGK) {
                        if (forced) step3<M_BGK, w, true, false, true>(p, parity, st);
                        else step3<M_BGK, w, false, false, true>(p, parity, st);
                    } else if (model == M_BGK_T) {
                        if (forced) step3<M_BGK_T, w, true, false, true>(p, parity, st);
                        else step3<M_BGK_T, w, false, false, true>(p, parity, st);
                    } else {
                        with_sc_model(model, [&](auto M) { step3<decltype(M)::value, w, true, false, true>(p, parity, st); });
                    }
                }
            });
        } else if (model == M_BGK) {
            bool v2 = false;
            if constexpr (sizeof(R) == 4) {
                if (forced != 2 && wmode <= 1 && p.bc[0] == 0 && p.nx % 2 == 0 && p.nx >= 64) {
                    // two cells per thread, vector accesses for the unshifted slots (k_step_v2); 128 threads = 256 cells of a row
                    int thr = 128;
                    while (thr > 32 && thr >= p.nx) thr /= 2;
                    const dim3 g((unsigned)((p.nx / 2 + thr - 1) / thr), (unsigned)p.ny, (unsigned)p.nz);
                    ok = with_int<2>(wmode, [&](auto W) {
                        with_int<2>(parity, [&](auto P) {
                            if (forced) k_step_v2<L, decltype(P)::value, decltype(W)::value, true><<<g, thr, 0, st>>>(p);
                            else k_step_v2<L, decltype(P)::value, decltype(W)::value, false><<<g, thr, 0, st>>>(p);
                        });
                    });
                    v2 = true;
                }
            }
            if (!v2)
                ok = with_int<3>(wmode, [&](auto W) {
                    constexpr int w = decltype(W)::value;
                    if (forced == 2) step3<M_BGK, w, true, true>(p, parity, st);
                    else if (forced) step3<M_BGK, w, true>(p, parity, st);
                    else step3<M_BGK, w, false>(p, parity, st);
                });
        } else if (model == M_BGK_T) {
            if (forced == 2) return cudaErrorInvalidValue;
            ok = with_int<3>(wmode, [&](auto W) {
                constexpr int w = decltype(W)::value;
                if (forced) step3<M_BGK_T, w, true>(p, parity, st);
                else step3<M_BGK_T, w, false>(p, parity, st);
            });
        } else {
            ok = with_sc_model(model, [&](auto M) {
                with_int<3>(wmode, [&](auto W) {
                    if (forced == 2) step3<decltype(M)::value, decltype(W)::value, true, true>(p, parity, st);
                    else step3<decltype(M)::value, decltype(W)::value, true>(p, parity, st);
                });
            });
        }
        return ok ? cudaGetLastError() : cudaErrorInvalidValue;
    }

    template <int MODEL>
    static void macros2(const KP<R>& p, int parity, int wmode, R* rho, R* u, R* phi, R* C, R* F, cudaStream_t st) {
        with_int<3>(wmode, [&](auto W) {
            with_int<2>(parity, [&](auto P) {
                k_macros<R, L, MODEL, decltype(P)::value, decltype(W)::value><<<grid_for(p), block_for(p), 0, st>>>(p, rho, u, phi, C, F);
            });
        });
    }
    static cudaError_t macros(const void* kp, int model, int parity, int wmode, void* rho, void* u, void* phi, void* C,
                              void* F, cudaStream_t st) {
        const KP<R>& p = *(const KP<R>*)kp;
        R *r = (R*)rho, *uu = (R*)u, *ph = (R*)phi, *c = (R*)C, *f = (R*)F;
        if (wmode < 0 || wmode > 2) return cudaErrorInvalidValue;
        if (model == M_BGK) macros2<M_BGK>(p, parity, wmode, r, uu, ph, c, f, st);
        else if (model == M_BGK_T) macros2<M_BGK_T>(p, parity, wmode, r, uu, ph, c, f, st);
        else if (!with_sc_model(model, [&](auto M) { macros2<decltype(M)::value>(p, parity, wmode, r, uu, ph, c, f, st); }))
            return cudaErrorInvalidValue;
        return cudaGetLastError();
    }

    template <class LL, bool TOC>
    static void permute2(const KP<R>& p, int parity, int wmode, R* slots, R* canon, int nl, cudaStream_t st, bool solid_lattice = false) {
        const dim3 g = grid_for(p);
        if (parity) {
            with_int<3>(wmode, [&](auto W) { k_permute<R, LL, 1, decltype(W)::value, TOC><<<g, block_for(p), 0, st>>>(p, slots, canon, nl, solid_lattice); });
        } else {
            k_permute<R, LL, 0, 0, TOC><<<g, block_for(p), 0, st>>>(p, slots, canon, nl, false);
        }
    }
    static cudaError_t permute(const void* kp, int model, int parity, int wmode, void* canon, int to_canonical,
                               cudaStream_t st) {
        using LS = typename ScalarOf<L>::type;
        const KP<R>& p = *(const KP<R>*)kp;
        const int S = (model == M_SC2 || model == M_SC2_ADE) ? 2 : 1;
        R* cf = (R*)canon;
        if (to_canonical) permute2<L, true>(p, parity, wmode, p.f, cf, S, st);
        else permute2<L, false>(p, parity, wmode, p.f, cf, S, st);
        if (model == M_SC2_ADE) {
            R* ch = cf + (size_t)S * L::Q * (size_t)p.N;
            if (to_canonical) permute2<LS, true>(p, parity, wmode, p.h, ch, 1, st);
            else permute2<LS, false>(p, parity, wmode, p.h, ch, 1, st);
        }
        if (model == M_BGK_T) {     // the internal-energy lattice lives on the flow lattice; solid nodes may carry it too (Eq. 31)
            R* ch = cf + (size_t)S * L::Q * (size_t)p.N;
            const bool sl = p.omega_s > (R)0;
            if (to_canonical) permute2<L, true>(p, parity, wmode, p.h, ch, 1, st, sl);
            else permute2<L, false>(p, parity, wmode, p.h, ch, 1, st, sl);
        }
        return cudaGetLastError();
    }

    static cudaError_t init(const void* kp, int model, const InitArgs* ia, cudaStream_t st) {
        const KP<R>& p = *(const KP<R>*)kp;
        const dim3 g = grid_for(p);
        switch (model) {
        case M_BGK: k_init<R, L, M_BGK><<<g, block_for(p), 0, st>>>(p, *ia); break;
        case M_SC1: k_init<R, L, M_SC1><<<g, block_for(p), 0, st>>>(p, *ia); break;
        case M_SC2: k_init<R, L, M_SC2><<<g, block_for(p), 0, st>>>(p, *ia); break;
        case M_SC2_ADE: k_init<R, L, M_SC2_ADE><<<g, block_for(p), 0, st>>>(p, *ia); break;
        case M_BGK_T: k_init<R, L, M_BGK_T><<<g, block_for(p), 0, st>>>(p, *ia); break;
        default: return cudaErrorInvalidValue;
        }
        return cudaGetLastError();
    }

    // resident-tile kernel (tile.cuh): wa == nullptr -> only return the number of co-resident blocks through *out_blocks
    template <int MODEL, bool WALLYZ, bool VSHIFT>
    static cudaError_t tile3(const KP<R>& p, int parity, const TileArgs* wa, int blocks, cudaStream_t st, int* out_blocks) {
        using C = TileCfg<R, L, MODEL>;
        constexpr size_t smem = C::SMEM;
        auto k0 = k_tile<R, L, MODEL, 0, WALLYZ, VSHIFT>;
        auto k1 = k_tile<R, L, MODEL, 1, WALLYZ, VSHIFT>;
        auto k = parity ? k1 : k0;
        // per device and context, cheap: set on every call
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        if (out_blocks) {
            int per_sm = 0, dev = 0, sms = 0;
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, C::THREADS, smem);
            if (e == cudaSuccess) e = cudaGetDevice(&dev);
            if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            if (e != cudaSuccess) return e;
            *out_blocks = per_sm * sms;
            return cudaSuccess;
        }
        // The psi parts wait for flags that other blocks set: all blocks must be co-resident.  The first launch of a
        // schedule (epoch 1) is a cooperative launch -- the runtime either makes the whole grid resident or refuses it --
        // which validates the block count; the later ones are plain launches of the same grid (a cooperative launch
        // costs about 0.4 ms per step on config 5)
        if (wa->epoch == 1) {
            void* args[2] = {(void*)&p, (void*)wa};
            return cudaLaunchCooperativeKernel((const void*)k, dim3((unsigned)blocks), dim3((unsigned)C::THREADS), args, smem, st);
        }
        k<<<blocks, C::THREADS, smem, st>>>(p, *wa);
        return cudaGetLastError();
    }
    static cudaError_t tile_any(const void* kp, int model, int parity, int walls, int vshift, const TileArgs* wa, int blocks, cudaStream_t st,
                                int* out_blocks) {
        const KP<R>& p = *(const KP<R>*)kp;
        cudaError_t e = cudaErrorInvalidValue;
        with_sc_model(model, [&](auto M) {
            constexpr int m = decltype(M)::value;
            if (walls) e = vshift ? tile3<m, true, true>(p, parity, wa, blocks, st, out_blocks) : tile3<m, true, false>(p, parity, wa, blocks, st, out_blocks);
            else e = vshift ? tile3<m, false, true>(p, parity, wa, blocks, st, out_blocks) : tile3<m, false, false>(p, parity, wa, blocks, st, out_blocks);
        });
        return e;
    }
    // vshift: the velocity-shift forcing scheme (Eq. 16-19) instead of Guo forcing
    static cudaError_t tile(const void* kp, int model, int parity, int walls, int vshift, const TileArgs* wa, int blocks, cudaStream_t st) {
        return tile_any(kp, model, parity, walls, vshift, wa, blocks, st, nullptr);
    }
    static int tile_blocks(int model, int parity, int walls, int vshift) {
        int b = 0;
        KP<R> dummy{};
        if (tile_any(&dummy, model, parity, walls, vshift, nullptr, 0, nullptr, &b) != cudaSuccess) { cudaGetLastError(); return 0; }
        return b;
    }
    static int tile_tx() { return TILE_ROW_BYTES / (int)sizeof(R); }

    static const Ops* ops() {
        static const Ops o = {&psi, &step, &macros, &permute, &init, &tile, &tile_blocks, &tile_tx};
        return &o;
    }
};

}  // namespace lbm
