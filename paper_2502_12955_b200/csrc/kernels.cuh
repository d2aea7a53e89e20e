// CUDA kernels of the lattice Boltzmann hot path (sm_100a).  See DESIGN.md for the data layout,
// the AA-pattern in-place streaming and the arithmetic specification.
//
// Layout (structure of arrays, ONE copy of the populations):
//   f[(sigma*Q + slot)*N + cell], h[slot*N + cell], psi[sigma*N + cell], cell = x + nx*(y + ny*z).
//
// AA-pattern in-place streaming: at time level t
//   t even: f_i(x,t) lives in slot i of cell x;
//   t odd : f_i(x,t) lives in slot opp(i) of cell x - c_i (periodic wrap), or, if x - c_i lies
//           beyond a bounce-back wall, in slot i of cell x itself.
// Call that location P_i(x).  One time step reads f_i from P_i(x), collides, and writes the
// post-collision f*_{opp(i)} back to the same P_i(x): every thread overwrites exactly the slots it
// read, slot sets of different cells are disjoint, so a step needs no barrier and no second copy.
// Eq. 5 and halfway bounce-back are both encoded in P_i.
//
// Arithmetic: the explicit-FMA expression tree of DESIGN.md section 5.  Every operation is a single IEEE-754
// add/sub/mul/div or, where the code says vfma, ONE fused multiply-add, in the context precision (the files are
// compiled with --fmad=false, default -prec-div=true, so nvcc forms no other FMA).  The per-cell code is generic in
// the value type V (vec.cuh): a scalar per thread, or two fp32 cells per thread in packed f32x2 instructions.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "lattice.cuh"
#include "vec.cuh"

namespace lbm {

enum { M_BGK = 0, M_SC1 = 1, M_SC2 = 2, M_SC2_ADE = 3, M_BGK_T = 4 };
enum { I_REST = 0, I_TAYLOR_GREEN = 1, I_DROPLET = 2, I_UNIFORM_NOISE = 3, I_RANDOM_DROPLETS = 4 };

constexpr int BLOCK = 256;   // largest block any kernel is launched with; the launchers pick blockDim.x (inst.cuh)

template <class R>
struct KP {
    R* f;
    R* h;
    R* psi;
    int nx, ny, nz, N;
    int bc[3];
    int psi_kind;
    R omega[2];               // 1/tau: Eq. 15
    R cfw[2][3];              // (1 - 1/(2 tau)) w_i per weight class (rest, axis, diagonal): prefactor of the Guo term, Eq. 15
    R tau[2];                 // tau itself (velocity-shift forcing, Eq. 16)
    R omega_c, inv_cs2g;      // 1/tau_c (Eq. 34), 1/c_{s,g}^2 = d/(1-w0) (Eq. 35, R6)
    R ws0, ws1;               // scalar-lattice weights
    R G[2][2];
    R G_ads[2];               // fluid-solid adhesion, Eq. 14
    R psi_wall;               // psi(rho_s) of the solid nodes in Eq. 12 (one component); used when solid_term != 0
    int solid_term;
    R wall_u[3][2][3];        // velocity of the wall at the low / high face of each axis (moving-wall bounce-back)
    const unsigned char* mask;  // solid-node mask (N bytes, non-zero = solid) or nullptr; read by the WALLS == 2 variants
    R rho0_psi;
    R force[3];
    R k_react;
    R omega_s, inv_rho_solid; // solid-phase internal-energy lattice on the solid nodes (M_BGK_T): 1/tau_{e,s} (0: none), 1/rho_s; Eq. 31-33
};

struct InitArgs {
    int kind;
    uint64_t seed;
    double rho_init[2], c_init, rho_in, rho_out, radius, width, noise_amp, u0;
    const double4* droplets;  // (cx, cy, cz, r), device
    int n_droplets;
};

template <int MODEL> struct ModelTraits {
    static constexpr int S = (MODEL == M_SC2 || MODEL == M_SC2_ADE) ? 2 : 1;
    static constexpr bool SC = MODEL == M_SC1 || MODEL == M_SC2 || MODEL == M_SC2_ADE;
    static constexpr bool SCALAR = MODEL == M_SC2_ADE;
    // internal-energy lattice g_i on the flow lattice (IEDDF, Eq. 27-30), stored in KP::h
    static constexpr bool THERMAL = MODEL == M_BGK_T;
};

// ------------------------------------------------------------------------------------------
// Thread mapping: grid (ceil(nx/blockDim.x), ny, nz), one block per segment of one x-row.  y and z are
// block-uniform, so the row bases of the 9 (cy,cz) neighbour rows (periodic wrap folded in) live
// in uniform registers; only x-1 / x / x+1 are per-thread.  An address is then
// (uniform slot base + uniform row base) + per-thread x: no integer division, one add per access.
// ------------------------------------------------------------------------------------------
// WALLS: 0 fully periodic; 1 bounce-back walls on the axes with bc = 1; 2 the same plus a solid-node mask
template <int D, int WALLS>
struct Nbr {
    static constexpr bool HAS_WALLS = WALLS != 0;
    int cell;              // x + nx*(y + ny*z)
    int xx[3];             // x-1, x, x+1 with periodic wrap (per thread)
    int ry[3], rz[3];      // nx*y', nx*ny*z' for y' = y-1,y,y+1 / z' = z-1,z,z+1 with wrap (uniform)
    bool lo[3], hi[3];
    unsigned blocked;      // bit (cx+1) + 3 (cy+1) + 9 (cz+1): the neighbour at that offset is a solid node of the mask
    bool solid;            // this cell is a solid node itself

    template <class R>
    __device__ __forceinline__ Nbr(const KP<R>& p, int x, int y, int z, bool solid_lattice = false) {
        const int nx = p.nx, ny = p.ny;
        xx[0] = (x == 0) ? nx - 1 : x - 1; xx[1] = x; xx[2] = (x == nx - 1) ? 0 : x + 1;
        ry[0] = ((y == 0) ? ny - 1 : y - 1) * nx; ry[1] = y * nx; ry[2] = ((y == ny - 1) ? 0 : y + 1) * nx;
        if constexpr (D == 3) {
            const int nz = p.nz, sxy = nx * ny;
            rz[0] = ((z == 0) ? nz - 1 : z - 1) * sxy; rz[1] = z * sxy; rz[2] = ((z == nz - 1) ? 0 : z + 1) * sxy;
        } else {
            rz[0] = rz[1] = rz[2] = 0;
        }
        cell = rz[1] + ry[1] + x;
        blocked = 0u;
        solid = false;
        if constexpr (WALLS) {
            lo[0] = p.bc[0] && x == 0; hi[0] = p.bc[0] && x == nx - 1;
            lo[1] = p.bc[1] && y == 0; hi[1] = p.bc[1] && y == ny - 1;
            lo[2] = D == 3 && p.bc[2] && z == 0; hi[2] = D == 3 && p.bc[2] && z == p.nz - 1;
            if constexpr (WALLS == 2) {
                // solid nodes of the mask reflect like a wall: one byte per lattice neighbour (L1 / L2 hits)
                solid = p.mask[cell] != 0;
                static_for<0, 27>([&](auto oc) {
                    constexpr int o = decltype(oc)::value;
                    constexpr int cx = o % 3 - 1, cy = (o / 3) % 3 - 1, cz = o / 9 - 1;
                    constexpr int n2 = cx * cx + cy * cy + cz * cz;
                    if constexpr ((D == 3 || cz == 0) && n2 >= 1 && n2 <= 2) {
                        if (p.mask[(rz[cz + 1] + ry[cy + 1]) + xx[cx + 1]]) blocked |= 1u << o;
                    }
                });
                // a solid node that carries the solid-phase lattice (Eq. 31): its neighbours must be solid nodes too,
                // the fluid nodes reflect (adiabatic interface) -- the same slot map with the roles exchanged
                if (solid && solid_lattice) blocked = ~blocked;
            }
        } else {
            lo[0] = lo[1] = lo[2] = hi[0] = hi[1] = hi[2] = false;
        }
    }
    // uniform part / per-thread part of the index of the cell at offset (cx,cy,cz)
    template <int CY, int CZ>
    __device__ __forceinline__ int row() const { return rz[CZ + 1] + ry[CY + 1]; }
    template <int CX>
    __device__ __forceinline__ int col() const { return xx[CX + 1]; }
    template <int CX, int CY, int CZ>
    __device__ __forceinline__ int at() const { return row<CY, CZ>() + col<CX>(); }
    // does the offset cross a bounce-back wall or end in a solid node?
    template <int CX, int CY, int CZ>
    __device__ __forceinline__ bool outside() const {
        if constexpr (!WALLS) return false;
        bool o = false;
        if constexpr (WALLS == 2) o = ((blocked >> ((CX + 1) + 3 * (CY + 1) + 9 * (CZ + 1))) & 1u) != 0u;
        if constexpr (CX < 0) o = o || lo[0];
        if constexpr (CX > 0) o = o || hi[0];
        if constexpr (CY < 0) o = o || lo[1];
        if constexpr (CY > 0) o = o || hi[1];
        if constexpr (CZ < 0) o = o || lo[2];
        if constexpr (CZ > 0) o = o || hi[2];
        return o;
    }
};

// the cell of this thread: false when the thread lies beyond the end of the row
__device__ __forceinline__ bool thread_cell(int nx, int& x, int& y, int& z) {
    x = blockIdx.x * blockDim.x + threadIdx.x; y = blockIdx.y; z = blockIdx.z;
    return x < nx;
}

// address of P_I(x): where f_I(x,t) is read and f*_{opp(I)}(x,t) is written.  The element index within one
// lattice (Q * N < 2^32, checked by lbm_create) is formed in 32 bits -- a uniform (slot, row) part plus the
// per-thread column -- so that an access costs one integer add and one IMAD.WIDE.
template <class L, int PARITY, int WALLS, int I, class R, class NB>
__device__ __forceinline__ R* slot_of(R* base, const NB& nb, size_t N) {
    const unsigned n = (unsigned)N;
    if constexpr (PARITY == 0 || I == 0) {
        return base + (((unsigned)I * n + (unsigned)nb.template row<0, 0>()) + (unsigned)nb.template col<0>());
    } else {
        constexpr int CX = -L::c(I, 0), CY = -L::c(I, 1), CZ = -L::c(I, 2);
        const unsigned nbr = ((unsigned)L::opp(I) * n + (unsigned)nb.template row<CY, CZ>()) + (unsigned)nb.template col<CX>();
        if constexpr (WALLS) {
            const unsigned own = ((unsigned)I * n + (unsigned)nb.template row<0, 0>()) + (unsigned)nb.template col<0>();
            return base + (nb.template outside<CX, CY, CZ>() ? own : nbr);
        } else {
            return base + nbr;
        }
    }
}

// sum_a c_{I,a} v_a in axis order, skipping the zero components (adding +-0 changes nothing).  (-x) + y is written
// y - x and (-x) - y as -(x + y): the same bits (negation is exact, addition commutes), one instruction less.
template <class L, int I, class V>
__device__ __forceinline__ V dotc(const V* v) {
    constexpr int c0 = L::c(I, 0), c1 = L::c(I, 1), c2 = L::D == 3 ? L::c(I, 2) : 0;
    constexpr int nnz = (c0 != 0) + (c1 != 0) + (c2 != 0);
    static_assert(nnz <= 2, "lattice velocities with at most two non-zero components");
    if constexpr (nnz == 0) {
        return vconst<V>(0.0);
    } else {
        constexpr int a = c0 != 0 ? 0 : (c1 != 0 ? 1 : 2);
        constexpr int sa = a == 0 ? c0 : (a == 1 ? c1 : c2);
        if constexpr (nnz == 1) {
            if constexpr (sa > 0) return v[a]; else return -v[a];
        } else {
            constexpr int b = (a == 0 && c1 != 0) ? 1 : 2;
            constexpr int sb = b == 1 ? c1 : c2;
            if constexpr (sa > 0 && sb > 0) return v[a] + v[b];
            else if constexpr (sa > 0) return v[a] - v[b];
            else if constexpr (sb > 0) return v[b] - v[a];
            else return -(v[a] + v[b]);
        }
    }
}

template <class L>
__host__ __device__ constexpr bool first_nonzero(int i, int a) {
    for (int k = 0; k < i; ++k)
        if (L::c(k, a) != 0) return false;
    return true;
}

// rho = sum_i f_i, j = sum_i c_i f_i, both in index order: Eq. 7-8 / 18
template <class L, class R>
__device__ __forceinline__ void moments(const R* fl, R& rho, R* j) {
    static_for<0, L::Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        if constexpr (i == 0) rho = fl[0]; else rho = rho + fl[i];
        static_for<0, L::D>([&](auto ac) {
            constexpr int a = decltype(ac)::value;
            constexpr int c = L::c(i, a);
            if constexpr (c != 0) {
                if constexpr (first_nonzero<L>(i, a)) j[a] = c > 0 ? fl[i] : -fl[i];
                else j[a] = c > 0 ? j[a] + fl[i] : j[a] - fl[i];
            }
        });
    });
}

template <class L, int PARITY, int WALLS, class R, class NB>
__device__ __forceinline__ void load_pops(R* __restrict__ base, const NB& nb, size_t N, R* fl) {
    static_for<0, L::Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        fl[i] = *slot_of<L, PARITY, WALLS, i>(base, nb, N);
    });
}
// writes fl[opp(i)] (post-collision) to P_i
template <class L, int PARITY, int WALLS, class R, class NB>
__device__ __forceinline__ void store_pops(R* __restrict__ base, const NB& nb, size_t N, const R* fl) {
    static_for<0, L::Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        *slot_of<L, PARITY, WALLS, i>(base, nb, N) = fl[L::opp(i)];
    });
}

// Shan-Chen stencil sums acc[t][a] = sum_{i>=1} w_i psi^t(x + c_i) c_{i,a}: Eq. 11 / 13
// COH: psi was written by other blocks of the SAME launch (wavefront kernel): read it from L2 (ld.global.cg),
// never from a possibly stale L1 line; otherwise through the read-only path
template <bool COH, class R>
__device__ __forceinline__ R load_psi(const R* q) {
    if constexpr (COH) return __ldcg(q); else return __ldg(q);
}

// acc[t][a] = fma(c_{i,a} w_i, psi^t(x + c_i), acc[t][a]) in index order from zero (row a3).
// Neighbours beyond a bounce-back wall are solid nodes: they are left out of the sum (Eq. 11-12: sum over FLUID
// neighbours; adding an exact zero instead of skipping changes no bit).
template <class L, int S, bool COH, class R, class NB>
__device__ __forceinline__ void sc_stencil(const R* __restrict__ psi, const NB& nb, size_t N, R (*acc)[3]) {
    static_for<0, S>([&](auto tc) {
        constexpr int t = decltype(tc)::value;
        const R* __restrict__ ps = psi + (size_t)t * N;
        acc[t][0] = acc[t][1] = acc[t][2] = (R)0;
        static_for<1, L::Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            constexpr int CX = L::c(i, 0), CY = L::c(i, 1), CZ = L::c(i, 2);
            R pv = load_psi<COH>(ps + ((unsigned)nb.template row<CY, CZ>() + (unsigned)nb.template col<CX>()));
            if (nb.template outside<CX, CY, CZ>()) pv = (R)0;       // fma(w, 0, acc) = acc: the term is left out
            static_for<0, L::D>([&](auto ac) {
                constexpr int a = decltype(ac)::value;
                constexpr int c = L::c(i, a);
                if constexpr (c != 0) acc[t][a] = vfma((R)(c * L::w(i)), pv, acc[t][a]);
            });
        });
    });
}

// adh[a] = sum_{i>=1} w_i s(x + c_i) c_{i,a}, s = 1 for the solid nodes beyond a wall: Eq. 14
template <class L, class R, class NB>
__device__ __forceinline__ void adhesion_sum(const NB& nb, R* adh) {
    adh[0] = adh[1] = adh[2] = (R)0;
    static_for<1, L::Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int CX = L::c(i, 0), CY = L::c(i, 1), CZ = L::c(i, 2);
        const R ws = nb.template outside<CX, CY, CZ>() ? (R)L::w(i) : (R)0;
        static_for<0, L::D>([&](auto ac) {
            constexpr int a = decltype(ac)::value;
            constexpr int c = L::c(i, a);
            if constexpr (c != 0) adh[a] = c > 0 ? adh[a] + ws : adh[a] - ws;
        });
    });
}

// ------------------------------------------------------------------------------------------
// per-cell state after steps a1-a4 (moments, force, barycentric velocity)
// ------------------------------------------------------------------------------------------
template <class R, class L, int MODEL>
struct CellMacro {
    static constexpr int S = ModelTraits<MODEL>::S;
    R rho[S];
    R j[S][3];
    R F[S][3];
    R u[3];
    R inv_rho;
};

// step a1: rho^s, j^s of every component (row a1)
template <class V, class L, int MODEL>
__device__ __forceinline__ void cell_moments(const V (*fl)[L::Q], CellMacro<V, L, MODEL>& m) {
    constexpr int S = ModelTraits<MODEL>::S;
    static_for<0, S>([&](auto sc) {
        constexpr int s = decltype(sc)::value;
        m.j[s][0] = m.j[s][1] = m.j[s][2] = vconst<V>(0.0);
        moments<L>(fl[s], m.rho[s], m.j[s]);
    });
}

// steps a3 (given the stencil sums), a4: force, barycentric velocity from the moments in m (rows a3-a4).
// acc[t][a] = sum_{i>=1} w_i psi^t(x + c_i) c_{i,a} and psi_own[s] = psi^s(x) are read only for Shan-Chen models.
// V: value type (scalar, or two fp32 cells), T: its scalar type.
template <class V, class L, int MODEL, bool FORCED, bool ADH = false, class T>
__device__ __forceinline__ void cell_force_velocity(const KP<T>& p, const V (*acc)[3], const V* psi_own,
                                                    CellMacro<V, L, MODEL>& m, const V* adh = nullptr) {
    constexpr int S = ModelTraits<MODEL>::S, D = L::D;
    constexpr bool SC = ModelTraits<MODEL>::SC;
    V (&j)[S][3] = m.j;
    V rho_t = m.rho[0];
    if constexpr (S == 2) rho_t = rho_t + m.rho[1];
    m.inv_rho = vrecip(rho_t);
    if constexpr (FORCED) {
        static_for<0, S>([&](auto sc) {
            constexpr int s = decltype(sc)::value;
            static_for<0, D>([&](auto ac) {
                constexpr int a = decltype(ac)::value;
                // constant body-force density, split by mass fraction for S = 2 (R5)
                V Fa = vbcast<V>(p.force[a]);
                if constexpr (S == 2) Fa = Fa * (m.rho[s] * m.inv_rho);
                if constexpr (SC) {
                    // Eq. 11 / 13: - psi^s(x) sum_t G_st acc^t
                    V t = vbcast<V>(p.G[s][0]) * acc[0][a];
                    if constexpr (S == 2) t = vfma(vbcast<V>(p.G[s][1]), acc[1][a], t);
                    Fa = vfma(-psi_own[s], t, Fa);
                    // fluid-solid adhesion at bounce-back walls, Eq. 14
                    if constexpr (ADH) Fa = vfma(-(vbcast<V>(p.G_ads[s]) * m.rho[s]), adh[a], Fa);
                    // solid term of Eq. 12, one component: -G psi(x) sum_solid w_i psi(rho_s) c_i
                    if constexpr (ADH && S == 1) {
                        if (p.solid_term) Fa = vfma(-(vbcast<V>(p.G[0][0]) * psi_own[0]), vbcast<V>(p.psi_wall) * adh[a], Fa);
                    }
                }
                m.F[s][a] = Fa;
            });
        });
    }
    // u^b = (1/rho) sum_sigma [ j^sigma + F^sigma / 2 ]: Eq. 20-21
    static_for<0, D>([&](auto ac) {
        constexpr int a = decltype(ac)::value;
        V jt = j[0][a];
        if constexpr (S == 2) jt = jt + j[1][a];
        if constexpr (FORCED) {
            V Ft = m.F[0][a];
            if constexpr (S == 2) Ft = Ft + m.F[1][a];
            m.u[a] = vfma(vconst<V>(0.5), Ft, jt) * m.inv_rho;
        } else {
            m.u[a] = jt * m.inv_rho;
        }
    });
}

// steps a1, a3 (given the stencil sums), a4 from the populations of the cell
template <class V, class L, int MODEL, bool FORCED, bool ADH = false, class T>
__device__ __forceinline__ void cell_macros_core(const KP<T>& p, const V (*fl)[L::Q], const V (*acc)[3], const V* psi_own,
                                                 CellMacro<V, L, MODEL>& m, const V* adh = nullptr) {
    cell_moments<V, L, MODEL>(fl, m);
    cell_force_velocity<V, L, MODEL, FORCED, ADH>(p, acc, psi_own, m, adh);
}

// Shan-Chen (velocity-shift) forcing scheme, DESIGN.md section 5 row a5': common velocity u' = sum_s (j^s / tau^s) /
// sum_s (rho^s / tau^s), Eq. 17; u^eq,s = u' + tau^s F^s / rho^s, Eq. 16
template <class V, class L, int MODEL, class T>
__device__ __forceinline__ void shift_velocities(const KP<T>& p, const CellMacro<V, L, MODEL>& m, V (*ueq)[3]) {
    constexpr int S = ModelTraits<MODEL>::S;
    V den = m.rho[0] * vbcast<V>(p.omega[0]);
    if constexpr (S == 2) den = vfma(m.rho[1], vbcast<V>(p.omega[1]), den);
    const V inv_den = vrecip(den);
    V inv_rs[S];
    static_for<0, S>([&](auto sc) { inv_rs[decltype(sc)::value] = vrecip(m.rho[decltype(sc)::value]); });
    static_for<0, L::D>([&](auto ac) {
        constexpr int a = decltype(ac)::value;
        V num = m.j[0][a] * vbcast<V>(p.omega[0]);
        if constexpr (S == 2) num = vfma(m.j[1][a], vbcast<V>(p.omega[1]), num);
        const V up = num * inv_den;
        static_for<0, S>([&](auto sc) {
            constexpr int s = decltype(sc)::value;
            ueq[s][a] = vfma(vbcast<V>(p.tau[s]) * m.F[s][a], inv_rs[s], up);
        });
    });
}

// steps a1-a4 given the populations of the cell (fl[s][i]) and the psi field in global memory
template <class R, class L, int MODEL, bool FORCED, bool COH = false, class NB>
__device__ __forceinline__ void cell_macros(const KP<R>& p, const NB& nb, const R (*fl)[L::Q], CellMacro<R, L, MODEL>& m) {
    constexpr int S = ModelTraits<MODEL>::S;
    constexpr bool SC = ModelTraits<MODEL>::SC;
    const size_t N = (size_t)p.N;
    R acc[S][3], psi_own[S], adh[3];
    constexpr bool ADH = FORCED && SC && NB::HAS_WALLS;
    if constexpr (FORCED && SC) {
        sc_stencil<L, S, COH>(p.psi, nb, N, acc);
        static_for<0, S>([&](auto sc) {
            constexpr int s = decltype(sc)::value;
            psi_own[s] = load_psi<COH>(p.psi + ((size_t)s * N + nb.cell));
        });
        if constexpr (ADH) adhesion_sum<L>(nb, adh);
    }
    cell_macros_core<R, L, MODEL, FORCED, ADH>(p, fl, acc, psi_own, m, adh);
}

// step a5 for one component: e_i = fma(3, cu, fma(4.5 cu, cu, base)), f^eq = (w rho) e_i (Eq. 6,
// PAPER.md:95, c_s^2 = 1/3); d = fma(-(w rho), e_i, f) = f - f^eq; f* = fma(-omega, d, f) (Eq. 15);
// Guo term (Eq. 22): Phi_i = fma(3, cF, fma(9 cu, cF, -3 u.F)), f* = fma((1 - 1/(2 tau)) w_i, Phi_i, f*).
// Opposite directions share cu, cF and the even terms (exactly: negation is exact).
// nomega = -1/tau; cfw[k] = (1 - 1/(2 tau)) w of weight class k (read only when FORCED).
template <class V, class L, bool FORCED>
__device__ __forceinline__ void collide(V* fl, V rho_s, const V* u, const V* Fs, V nomega, const V* cfw) {
    constexpr int D = L::D;
    V usq = u[0] * u[0];
    usq = vfma(u[1], u[1], usq);
    if constexpr (D == 3) usq = vfma(u[2], u[2], usq);
    const V base = vfma(vconst<V>(-1.5), usq, vconst<V>(1.0));
    V m3uF = vconst<V>(0.0);
    if constexpr (FORCED) {
        V uF = u[0] * Fs[0];
        uF = vfma(u[1], Fs[1], uF);
        if constexpr (D == 3) uF = vfma(u[2], Fs[2], uF);
        m3uF = vconst<V>(-3.0) * uF;
    }
    // -(w rho) per weight class
    const V nwr[3] = {vconst<V>(-L::w(0)) * rho_s, vconst<V>(-L::w(1)) * rho_s, vconst<V>(-L::w(L::Q - 1)) * rho_s};
    const V c3 = vconst<V>(3.0), cm3 = vconst<V>(-3.0);
    {   // rest population: c = 0, e_0 = base, Phi_0 = -3 u.F
        V fs = vfma(nomega, vfma(nwr[0], base, fl[0]), fl[0]);
        if constexpr (FORCED) fs = vfma(cfw[0], m3uF, fs);
        fl[0] = fs;
    }
    static_for<1, L::Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int o = L::opp(i);
        if constexpr (i < o) {
            constexpr int k = L::wclass(i);
            const V cu = dotc<L, i>(u);
            const V bq = vfma(vconst<V>(4.5) * cu, cu, base);
            const V e_i = vfma(c3, cu, bq);
            const V e_o = vfma(cm3, cu, bq);
            V fs_i = vfma(nomega, vfma(nwr[k], e_i, fl[i]), fl[i]);
            V fs_o = vfma(nomega, vfma(nwr[k], e_o, fl[o]), fl[o]);
            if constexpr (FORCED) {
                const V cF = dotc<L, i>(Fs);
                const V A = vfma(vconst<V>(9.0) * cu, cF, m3uF);
                fs_i = vfma(cfw[k], vfma(c3, cF, A), fs_i);
                fs_o = vfma(cfw[k], vfma(cm3, cF, A), fs_o);
            }
            fl[i] = fs_i;
            fl[o] = fs_o;
        }
    });
}

// step a6: scalar lattice, Eq. 34-36 + source w_i R, R = -k C 4 rhoA rhoB/(rhoA+rhoB)^2 (R8):
// d = fma(-(w C), fma(1/c_sg^2, c.u, 1), h) = h - h^eq;  h* = fma(w, R, fma(-omega_c, d, h))
template <class V, class LS, class T>
__device__ __forceinline__ void collide_scalar(const KP<T>& p, V* hl, V rA, V rB, V inv_rho, const V* u) {
    V C = hl[0];
    static_for<1, LS::Q>([&](auto ic) { C = C + hl[decltype(ic)::value]; });
    const V chi = (vconst<V>(4.0) * (rA * inv_rho)) * (rB * inv_rho);
    const V Rsrc = -((vbcast<V>(p.k_react) * C) * chi);
    const V nwC0 = vbcast<V>(-p.ws0) * C, nwC1 = vbcast<V>(-p.ws1) * C;
    const V w0 = vbcast<V>(p.ws0), w1 = vbcast<V>(p.ws1), nomc = vbcast<V>(-p.omega_c);
    const V inv = vbcast<V>(p.inv_cs2g), ninv = vbcast<V>(-p.inv_cs2g), one = vconst<V>(1.0);
    hl[0] = vfma(w0, Rsrc, vfma(nomc, hl[0] + nwC0, hl[0]));       // c = 0: h^eq = (w_0 C) * 1 exactly
    static_for<1, LS::Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int o = LS::opp(i);
        if constexpr (i < o) {
            const V m = dotc<LS, i>(u);
            const V d_i = vfma(nwC1, vfma(inv, m, one), hl[i]);
            const V d_o = vfma(nwC1, vfma(ninv, m, one), hl[o]);
            hl[i] = vfma(w1, Rsrc, vfma(nomc, d_i, hl[i]));
            hl[o] = vfma(w1, Rsrc, vfma(nomc, d_o, hl[o]));
        }
    });
}

// step a5 for component s with the constants of the context (KP): -omega^s and (1 - 1/(2 tau^s)) w_k
template <class V, class L, bool FORCED, int s, class T>
__device__ __forceinline__ void collide_component(const KP<T>& p, V* fl, V rho_s, const V* u, const V* Fs) {
    const V cfw[3] = {vbcast<V>(p.cfw[s][0]), vbcast<V>(p.cfw[s][1]), vbcast<V>(p.cfw[s][2])};
    collide<V, L, FORCED>(fl, rho_s, u, Fs, vbcast<V>(-p.omega[s]), cfw);
}

// ------------------------------------------------------------------------------------------
// psi pass (step a2): rho^sigma from the populations at the current parity, psi^sigma to HBM
// ------------------------------------------------------------------------------------------
// psi^sigma of the cell (x,y,z) at the current parity
template <class R, class L, int MODEL, int PARITY, int WALLS = false>
__device__ __forceinline__ void psi_cell(const KP<R>& p, int x, int y, int z) {
    constexpr int S = ModelTraits<MODEL>::S, Q = L::Q;
    const size_t N = (size_t)p.N;
    const Nbr<L::D, WALLS> nb(p, x, y, z);
    const int cell = nb.cell;
    if (WALLS == 2 && nb.solid) return;
    static_for<0, S>([&](auto sc) {
        constexpr int s = decltype(sc)::value;
        R fl[Q];
        load_pops<L, PARITY, WALLS>(p.f + (size_t)s * Q * N, nb, N, fl);
        R rho, j[3];
        moments<L>(fl, rho, j);
        p.psi[(size_t)s * N + cell] = psi_of(rho, p.psi_kind, p.rho0_psi);
    });
}

template <class R, class L, int MODEL, int PARITY, int WALLS = false>
__global__ void __launch_bounds__(BLOCK) k_psi(const __grid_constant__ KP<R> p) {
    int x, y, z;
    if (!thread_cell(p.nx, x, y, z)) return;
    psi_cell<R, L, MODEL, PARITY, WALLS>(p, x, y, z);
}

// ------------------------------------------------------------------------------------------
// fused step (a1, a3-a8): one thread per cell
// ------------------------------------------------------------------------------------------
// Moving-wall halfway bounce-back (DESIGN R24): a post-collision population f*_k that leaves the
// cell through a wall comes back as f_opp(k) minus 2 w_k rho (c_k . u_w) / c_s^2.  It is stored exactly once (to
// P_opp(k)(x), the cell's own slot), so the correction is applied to the register value before the stores.
// u_w: the first wall axis (x, y, z order) the direction crosses.
template <class L, class R, class NB>
__device__ __forceinline__ void moving_wall_correction(const KP<R>& p, const NB& nb, R rho_s, R* fl) {
    static_for<1, L::Q>([&](auto kc) {
        constexpr int k = decltype(kc)::value;
        constexpr int CX = L::c(k, 0), CY = L::c(k, 1), CZ = L::c(k, 2);
        if (nb.template outside<CX, CY, CZ>()) {
            const R zero[3] = {(R)0, (R)0, (R)0};   // a solid node of the mask is at rest
            const R* uw = zero;
            bool found = false;
            if constexpr (CX != 0) { if (CX < 0 ? nb.lo[0] : nb.hi[0]) { uw = p.wall_u[0][CX < 0 ? 0 : 1]; found = true; } }
            if constexpr (CY != 0) { if (!found && (CY < 0 ? nb.lo[1] : nb.hi[1])) { uw = p.wall_u[1][CY < 0 ? 0 : 1]; found = true; } }
            if constexpr (CZ != 0) { if (!found && (CZ < 0 ? nb.lo[2] : nb.hi[2])) { uw = p.wall_u[2][CZ < 0 ? 0 : 1]; found = true; } }
            const R u3[3] = {uw[0], uw[1], uw[2]};
            const R cuw = dotc<L, k>(u3);
            fl[k] = vfma(-((R)(6.0 * L::w(k)) * rho_s), cuw, fl[k]);
        }
    });
}

// one cell of the fused step (k_step)
template <class R, class L, int MODEL, int PARITY, int WALLS, bool FORCED, bool COH = false, bool VSHIFT = false, bool MOVING = false>
__device__ __forceinline__ void step_cell(const KP<R>& p, int x, int y, int z) {
    using MT = ModelTraits<MODEL>;
    using LS = typename ScalarOf<L>::type;
    constexpr int S = MT::S, Q = L::Q;
    const size_t N = (size_t)p.N;
    const bool solid_lattice = MT::THERMAL && WALLS == 2 && p.omega_s > (R)0;
    const Nbr<L::D, WALLS> nb(p, x, y, z, solid_lattice);
    if (WALLS == 2 && nb.solid) {                    // solid nodes are not updated ...
        if constexpr (MT::THERMAL && WALLS == 2) {
            if (solid_lattice) {
                // ... except for the solid-phase internal-energy lattice, Eq. 31: g^eq_{s,i} = w_i rho_s eps_s
                // (Eq. 32) with rho_s eps_s = sum_i g_{s,i} (Eq. 33); streams among solid nodes, reflected by fluid nodes
                R gl[Q];
                load_pops<L, PARITY, WALLS>(p.h, nb, N, gl);
                R E = gl[0];
                static_for<1, Q>([&](auto ic) { E = E + gl[decltype(ic)::value]; });
                static_for<0, Q>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    gl[i] = vfma(-p.omega_s, vfma((R)(-L::w(i)), E, gl[i]), gl[i]);
                });
                Nbr<L::D, WALLS> ns = nb;
                asm volatile("" : "+r"(ns.xx[0]), "+r"(ns.xx[1]), "+r"(ns.xx[2]));
                store_pops<L, PARITY, WALLS>(p.h, ns, N, gl);
            }
        }
        return;
    }

    R fl[S][Q];
    static_for<0, S>([&](auto sc) {
        constexpr int s = decltype(sc)::value;
        load_pops<L, PARITY, WALLS>(p.f + (size_t)s * Q * N, nb, N, fl[s]);
    });
    R hl[LS::Q];
    if constexpr (MT::SCALAR) load_pops<LS, PARITY, WALLS>(p.h, nb, N, hl);
    R gl[Q];
    if constexpr (MT::THERMAL) load_pops<L, PARITY, WALLS>(p.h, nb, N, gl);

    CellMacro<R, L, MODEL> m;
    cell_macros<R, L, MODEL, FORCED, COH>(p, nb, fl, m);

    // Shan-Chen (velocity-shift) forcing scheme: common velocity u' = sum_s (j^s / tau^s) / sum_s (rho^s / tau^s),
    // Eq. 17; u^eq,s = u' + tau^s F^s / rho^s, Eq. 16; no forcing term F_i
    R ueq[S][3];
    if constexpr (VSHIFT) shift_velocities<R, L, MODEL>(p, m, ueq);

    Nbr<L::D, WALLS> ns = nb;
    asm volatile("" : "+r"(ns.xx[0]), "+r"(ns.xx[1]), "+r"(ns.xx[2]));
    static_for<0, S>([&](auto sc) {
        constexpr int s = decltype(sc)::value;
        if constexpr (VSHIFT) collide_component<R, L, false, s>(p, fl[s], m.rho[s], ueq[s], m.F[s]);
        else collide_component<R, L, FORCED, s>(p, fl[s], m.rho[s], m.u, m.F[s]);
        if constexpr (MOVING && WALLS) moving_wall_correction<L>(p, nb, m.rho[s], fl[s]);
        store_pops<L, PARITY, WALLS>(p.f + (size_t)s * Q * N, ns, N, fl[s]);
    });
    if constexpr (MT::SCALAR) {
        collide_scalar<R, LS>(p, hl, m.rho[0], m.rho[S - 1], m.inv_rho, m.u);
        store_pops<LS, PARITY, WALLS>(p.h, ns, N, hl);
    }
    if constexpr (MT::THERMAL) {
        // Eq. 27 with g^eq = w_i (rho eps) [1 + 3 cu + 4.5 cu^2 - 1.5 u.u] (Eq. 30), rho eps = sum_i g_i (Eq. 29):
        // the LBGK relaxation of Eq. 6 with sum g in place of rho and tau_e in place of tau; reflected at walls
        R E = gl[0];
        static_for<1, Q>([&](auto ic) { E = E + gl[decltype(ic)::value]; });
        collide<R, L, false>(gl, E, m.u, m.F[0], -p.omega_c, (const R*)nullptr);
        store_pops<L, PARITY, WALLS>(p.h, ns, N, gl);
    }
}

// k_step always runs with 128 threads.  The minimum number of resident blocks per SM bounds its registers
// (ptxas fills whatever the bound leaves: a bound of 1 block made fp64 BGK use 168 registers instead of 80).
// Measured on cfg4: fp32 10 or 12 blocks 41.4 GLUPS, 8: 39.4, 16: 36.0; fp64 4-6 blocks 22.1, 8: 21.3.
#ifndef LBM_MINB_BGK32
#define LBM_MINB_BGK32 10
#endif
#ifndef LBM_MINB_BGK64
#define LBM_MINB_BGK64 6
#endif
template <class R, int MODEL, int Q = 9> struct StepBounds {
    static constexpr int THREADS = 128;
    // two-component D3Q19 in fp64 holds 2 x 19 doubles per thread: 3 blocks (170 registers) avoid the spills of 5
    static constexpr int MINB = MODEL == M_BGK ? (sizeof(R) == 4 ? LBM_MINB_BGK32 : LBM_MINB_BGK64)
                              : (MODEL == M_SC1 ? 6 : (sizeof(R) == 8 && Q == 19 ? 3 : 5));
};

template <class R, class L, int MODEL, int PARITY, int WALLS, bool FORCED, bool VSHIFT = false, bool MOVING = false>
__global__ void __launch_bounds__(StepBounds<R, MODEL, L::Q>::THREADS, StepBounds<R, MODEL, L::Q>::MINB) k_step(const __grid_constant__ KP<R> p) {
    int x, y, z;
    if (!thread_cell(p.nx, x, y, z)) return;
    step_cell<R, L, MODEL, PARITY, WALLS, FORCED, false, VSHIFT, MOVING>(p, x, y, z);
}

// ------------------------------------------------------------------------------------------
// fused fp32 BGK step, TWO cells (x, x+1) per thread in packed f32x2 arithmetic (V = F2: one FADD2 / FMUL2 / FFMA2
// per operation of the expression tree for both cells).  Slots that are not shifted in x (all of them at even
// parity, those with c_x = 0 at odd parity) are moved as one 8-byte access per thread -- the loaded register pair IS
// the packed operand -- the others element-wise.  Same per-cell arithmetic as k_step, bit for bit.  Needs an even nx
// and periodic x (the launcher checks).  k_step in fp32 is limited by instruction issue; in fp64 there is no packed
// arithmetic and the single-cell kernel is at the copy peak anyway.
// ------------------------------------------------------------------------------------------
template <class L, int PARITY, int WALLS, bool FORCED>
__global__ void __launch_bounds__(128, 6) k_step_v2(const __grid_constant__ KP<float> p) {
    constexpr int Q = L::Q;
    const int x = 2 * (int)(blockIdx.x * blockDim.x + threadIdx.x), y = (int)blockIdx.y, z = (int)blockIdx.z;
    if (x >= p.nx) return;
    const size_t N = (size_t)p.N;
    const Nbr<L::D, WALLS> na(p, x, y, z), nbb(p, x + 1, y, z);
    F2 f2[1][Q];
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        float* pa = slot_of<L, PARITY, WALLS, i>(p.f, na, N);
        if constexpr (PARITY == 0 || L::c(i, 0) == 0) f2[0][i].v = *reinterpret_cast<const unsigned long long*>(pa);
        else f2[0][i] = pack2(*pa, *slot_of<L, PARITY, WALLS, i>(p.f, nbb, N));
    });
    CellMacro<F2, L, M_BGK> m;
    cell_macros_core<F2, L, M_BGK, FORCED>(p, f2, (const F2(*)[3])nullptr, (const F2*)nullptr, m);
    collide_component<F2, L, FORCED, 0>(p, f2[0], m.rho[0], m.u, m.F[0]);
    Nbr<L::D, WALLS> sa = na, sb = nbb;
    asm volatile("" : "+r"(sa.xx[0]), "+r"(sa.xx[1]), "+r"(sa.xx[2]), "+r"(sb.xx[0]), "+r"(sb.xx[1]), "+r"(sb.xx[2]));
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        float* pa = slot_of<L, PARITY, WALLS, i>(p.f, sa, N);
        if constexpr (PARITY == 0 || L::c(i, 0) == 0) {
            *reinterpret_cast<unsigned long long*>(pa) = f2[0][L::opp(i)].v;
        } else {
            float lo, hi;
            unpack2(f2[0][L::opp(i)], lo, hi);
            *pa = lo;
            *slot_of<L, PARITY, WALLS, i>(p.f, sb, N) = hi;
        }
    });
}

// ------------------------------------------------------------------------------------------
// macros out (step a9) and force diagnostic; psi must be current
// ------------------------------------------------------------------------------------------
template <class R, class L, int MODEL, int PARITY, int WALLS>
__global__ void __launch_bounds__(BLOCK) k_macros(const __grid_constant__ KP<R> p, R* __restrict__ rho_o,
                                                  R* __restrict__ u_o, R* __restrict__ phi_o, R* __restrict__ C_o,
                                                  R* __restrict__ F_o) {
    using MT = ModelTraits<MODEL>;
    using LS = typename ScalarOf<L>::type;
    constexpr int S = MT::S, Q = L::Q, D = L::D;
    int x, y, z;
    if (!thread_cell(p.nx, x, y, z)) return;
    const size_t N = (size_t)p.N;
    const bool solid_lattice = MT::THERMAL && WALLS == 2 && p.omega_s > (R)0;
    const Nbr<D, WALLS> nb(p, x, y, z, solid_lattice);
    const int cell = nb.cell;
    if (WALLS == 2 && nb.solid) {        // no fluid here: every field reads as zero
        if (rho_o) static_for<0, S>([&](auto sc) { rho_o[(size_t)decltype(sc)::value * N + cell] = (R)0; });
        if (u_o) static_for<0, D>([&](auto ac) { u_o[(size_t)decltype(ac)::value * N + cell] = (R)0; });
        if (phi_o) phi_o[cell] = (R)0;
        if (C_o) {
            R eps_s = (R)0;
            if constexpr (MT::THERMAL && WALLS == 2) {
                if (solid_lattice) {     // eps_s = sum_i g_{s,i} / rho_s, Eq. 33
                    R gl[Q];
                    load_pops<L, PARITY, WALLS>(p.h, nb, N, gl);
                    R E = gl[0];
                    static_for<1, Q>([&](auto ic) { E = E + gl[decltype(ic)::value]; });
                    eps_s = E * p.inv_rho_solid;
                }
            }
            C_o[cell] = eps_s;
        }
        if (F_o) static_for<0, S * D>([&](auto kc) { F_o[(size_t)decltype(kc)::value * N + cell] = (R)0; });
        return;
    }
    R fl[S][Q];
    static_for<0, S>([&](auto sc) {
        constexpr int s = decltype(sc)::value;
        load_pops<L, PARITY, WALLS>(p.f + (size_t)s * Q * N, nb, N, fl[s]);
    });
    CellMacro<R, L, MODEL> m;
    cell_macros<R, L, MODEL, true>(p, nb, fl, m);
    if (rho_o) static_for<0, S>([&](auto sc) { rho_o[(size_t)decltype(sc)::value * N + cell] = m.rho[decltype(sc)::value]; });
    if (u_o) static_for<0, D>([&](auto ac) { u_o[(size_t)decltype(ac)::value * N + cell] = m.u[decltype(ac)::value]; });
    if (phi_o) {
        if constexpr (S == 2) phi_o[cell] = (m.rho[0] - m.rho[1]) * m.inv_rho;
        else if constexpr (MT::SC) phi_o[cell] = p.psi[cell];
        else phi_o[cell] = psi_of(m.rho[0], p.psi_kind, p.rho0_psi);
    }
    if constexpr (MT::SCALAR) {
        if (C_o) {
            R hl[LS::Q];
            load_pops<LS, PARITY, WALLS>(p.h, nb, N, hl);
            R C = hl[0];
            static_for<1, LS::Q>([&](auto ic) { C = C + hl[decltype(ic)::value]; });
            C_o[cell] = C;
        }
    }
    if constexpr (MT::THERMAL) {
        if (C_o) {      // internal energy eps = sum_i g_i / rho, Eq. 29
            R gl[Q];
            load_pops<L, PARITY, WALLS>(p.h, nb, N, gl);
            R E = gl[0];
            static_for<1, Q>([&](auto ic) { E = E + gl[decltype(ic)::value]; });
            C_o[cell] = E * m.inv_rho;
        }
    }
    if (F_o)
        static_for<0, S>([&](auto sc) {
            constexpr int s = decltype(sc)::value;
            static_for<0, D>([&](auto ac) {
                constexpr int a = decltype(ac)::value;
                F_o[((size_t)s * D + a) * N + cell] = m.F[s][a];
            });
        });
}

// canonical populations f_i(x,t) out of the slot array at the current parity (and back)
template <class R, class L, int PARITY, int WALLS, bool TO_CANONICAL>
__global__ void __launch_bounds__(BLOCK) k_permute(const __grid_constant__ KP<R> p, R* __restrict__ slots,
                                                   R* __restrict__ canon, int n_lattices, bool solid_lattice) {
    int x, y, z;
    if (!thread_cell(p.nx, x, y, z)) return;
    const size_t N = (size_t)p.N;
    const Nbr<L::D, WALLS> nb(p, x, y, z, WALLS == 2 && solid_lattice);   // solid_lattice: the solid nodes carry this lattice too (Eq. 31)
    const int cell = nb.cell;
    for (int s = 0; s < n_lattices; ++s) {
        R* sb = slots + (size_t)s * L::Q * N;
        R* cb = canon + (size_t)s * L::Q * N;
        static_for<0, L::Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            R* P = slot_of<L, PARITY, WALLS, i>(sb, nb, N);
            if (WALLS == 2 && nb.solid && !solid_lattice) P = sb + ((size_t)i * N + cell);      // an inert solid node keeps its values in its own slots
            if constexpr (TO_CANONICAL) cb[(size_t)i * N + cell] = *P;
            else *P = cb[(size_t)i * N + cell];
        });
    }
}

// ------------------------------------------------------------------------------------------
// seeded initial condition: macroscopic fields in double, then
// equilibrium populations (Eq. 6) in R, written at even parity
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint64_t mix64(uint64_t z) {   // splitmix64 finaliser
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
__device__ __forceinline__ double uniform01(uint64_t seed, uint64_t index) {
    const uint64_t hsh = mix64(seed + 0x9E3779B97F4A7C15ULL * (index + 1ULL));
    return (double)(hsh >> 11) * (1.0 / 9007199254740992.0);
}
__device__ __forceinline__ double min_image(double a, double b, int n, int bc) {
    double dd = fabs(a - b);
    if (bc == 0 && (double)n - dd < dd) dd = (double)n - dd;
    return dd;
}

template <class R, class L, int MODEL>
__global__ void __launch_bounds__(BLOCK) k_init(const __grid_constant__ KP<R> p, const __grid_constant__ InitArgs ia) {
    using MT = ModelTraits<MODEL>;
    using LS = typename ScalarOf<L>::type;
    constexpr int S = MT::S, Q = L::Q, D = L::D;
    int x, y, z;
    if (!thread_cell(p.nx, x, y, z)) return;
    const size_t N = (size_t)p.N;
    const int nx = p.nx, ny = p.ny, nz = p.nz;
    const int cell = x + nx * (y + ny * z);
    const double PI = 3.14159265358979323846;
    double r0[2] = {ia.rho_init[0], ia.rho_init[1]};
    double u0[3] = {0.0, 0.0, 0.0};
    double c0 = ia.c_init;
    if (ia.kind == I_TAYLOR_GREEN) {
        if constexpr (D == 2) {
            // planar Taylor-Green vortex (R19), the 2D analogue of Eq. 45
            const double kx = 2.0 * PI / (double)nx, ky = 2.0 * PI / (double)ny;
            const double A = ia.u0, B = ia.u0 * (kx / ky);
            u0[0] = -A * cos(kx * x) * sin(ky * y);
            u0[1] = B * sin(kx * x) * cos(ky * y);
            r0[0] = ia.rho_init[0] * (1.0 - 0.75 * (A * A * cos(2.0 * kx * x) + B * B * cos(2.0 * ky * y)));
        } else {
            // Eq. 45a-c; pressure: textbook form (R21); rho = rho0 + 3 (P - P0)
            const double kx = 2.0 * PI / (double)nx, ky = 2.0 * PI / (double)ny, kz = 2.0 * PI / (double)nz;
            u0[0] = ia.u0 * cos(kx * x) * sin(ky * y) * sin(kz * z);
            u0[1] = -ia.u0 * sin(kx * x) * cos(ky * y) * sin(kz * z);
            u0[2] = 0.0;
            r0[0] = ia.rho_init[0] * (1.0 + 3.0 * (ia.u0 * ia.u0 / 16.0) * (cos(2.0 * kz * z) + 2.0) *
                                                (cos(2.0 * kx * x) + cos(2.0 * ky * y)));
        }
    } else if (ia.kind == I_DROPLET) {
        // centred droplet with a tanh profile of width W (R17), then seeded noise (R16)
        const double ddx = min_image((double)x, 0.5 * (nx - 1), nx, p.bc[0]);
        const double ddy = min_image((double)y, 0.5 * (ny - 1), ny, p.bc[1]);
        const double ddz = (D == 3) ? min_image((double)z, 0.5 * (nz - 1), nz, p.bc[2]) : 0.0;
        const double dist = sqrt(ddx * ddx + ddy * ddy + ddz * ddz);
        const double th = tanh(2.0 * (dist - ia.radius) / ia.width);
        const double mean = 0.5 * (ia.rho_in + ia.rho_out), half = 0.5 * (ia.rho_in - ia.rho_out);
        r0[0] = mean - half * th;
        r0[1] = mean + half * th;
        c0 = ia.c_init * (0.5 * (1.0 - th));
        for (int s = 0; s < S; ++s)
            r0[s] = r0[s] * (1.0 + ia.noise_amp * (2.0 * uniform01(ia.seed, (uint64_t)cell + (uint64_t)N * s) - 1.0));
    } else if (ia.kind == I_UNIFORM_NOISE) {
        for (int s = 0; s < S; ++s)
            r0[s] = ia.rho_init[s] * (1.0 + ia.noise_amp * (2.0 * uniform01(ia.seed, (uint64_t)cell + (uint64_t)N * s) - 1.0));
    } else if (ia.kind == I_RANDOM_DROPLETS) {
        // indicator I = max_k prof((dist_k - r_k)/W), prof = cubic smoothstep (R18)
        double I = 0.0;
        for (int k = 0; k < ia.n_droplets; ++k) {
            const double4 dr = ia.droplets[k];
            const double ddx = min_image((double)x, dr.x, nx, p.bc[0]);
            const double ddy = min_image((double)y, dr.y, ny, p.bc[1]);
            const double ddz = (D == 3) ? min_image((double)z, dr.z, nz, p.bc[2]) : 0.0;
            const double s = (sqrt(ddx * ddx + ddy * ddy + ddz * ddz) - dr.w) / ia.width;
            const double v = (s <= -1.0) ? 1.0 : (s >= 1.0 ? 0.0 : (0.5 - 0.75 * s) + (0.25 * s) * (s * s));
            if (v > I) I = v;
        }
        r0[0] = ia.rho_out + (ia.rho_in - ia.rho_out) * I;
        r0[1] = ia.rho_in - (ia.rho_in - ia.rho_out) * I;
        c0 = ia.c_init * I;
    }
    // populations = equilibrium at (rho, u), no non-equilibrium part (R10)
    const R u[3] = {(R)u0[0], (R)u0[1], (R)u0[2]};
    R usq = u[0] * u[0];
    usq = vfma(u[1], u[1], usq);
    if constexpr (D == 3) usq = vfma(u[2], u[2], usq);
    const R base = vfma((R)-1.5, usq, (R)1);
    static_for<0, S>([&](auto sc) {
        constexpr int s = decltype(sc)::value;
        const R rho_s = (R)r0[s];
        R* fb = p.f + (size_t)s * Q * N;
        static_for<0, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            const R cu = dotc<L, i>(u);
            fb[(size_t)i * N + cell] = ((R)L::w(i) * rho_s) * vfma((R)3, cu, vfma((R)4.5 * cu, cu, base));
        });
    });
    if constexpr (MT::SCALAR) {
        static_for<0, LS::Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            const R cu = dotc<LS, i>(u);
            const R wsi = i == 0 ? p.ws0 : p.ws1;
            p.h[(size_t)i * N + cell] = (wsi * (R)c0) * vfma(p.inv_cs2g, cu, (R)1);
        });
    }
    if constexpr (MT::THERMAL) {     // g_i = g^eq(rho eps, u), eps = c_init: Eq. 30
        const R rhoE = (R)r0[0] * (R)c0;
        static_for<0, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            const R cu = dotc<L, i>(u);
            p.h[(size_t)i * N + cell] = ((R)L::w(i) * rhoE) * vfma((R)3, cu, vfma((R)4.5 * cu, cu, base));
        });
    }
}

}  // namespace lbm
