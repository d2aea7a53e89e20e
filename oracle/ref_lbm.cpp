/*
 * oracle/ref_lbm.cpp -- the CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded, two-buffer ("double-population")
 * implementation of the lattice Boltzmann update of CooLBM (arXiv 2502.12955):
 * it follows the paper step by step, in the paper's order and notation, one
 * full-field loop per step, with no blocking, fusion or in-place tricks.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may use it.  It shares no code with the CUDA library
 * in paper_2502_12955_b200/ and neither includes the other.
 *
 * Citations are PAPER.md line numbers + equation.  "DESIGN R<n>" refers to the
 * numbered readings of the paper listed in DESIGN.md.
 *
 * Parity pins (tests/test_oracle_*.py, all "-m 'not gpu'"):
 *   Taylor-Green decay exp(-2 nu k^2 t); Poiseuille parabola + halfway-BB slip;
 *   uniform-force momentum growth; mass / momentum invariants; Shan-Chen force
 *   against the literal pair sum of Eq. 9; Laplace law; flat-interface pressure
 *   balance Eq. 46; demixing threshold; scalar diffusion / advection / reaction
 *   closed forms; equilibrium moments; rotation equivariance; lattice tables
 *   against tests/golden/.  Nothing in this file is "parity unpinned".
 *
 * Arithmetic ("explicit-FMA specification"): every operation
 * below is a single IEEE-754 add, sub, mul, div or fused multiply-add in the
 * context precision R (float or double), evaluated exactly as parenthesised.
 * A product that feeds a sum is fused into it where -- and only where -- the code
 * says std::fma (one rounding for a*b + c); build with -ffp-contract=off so the
 * compiler forms no other FMA.  Constants are formed in double from the double
 * parameters and rounded once to R.
 */
#include "ref_lbm.h"

#include <cmath>
#include <cstdint>
#include <cstring>
#include <new>
#include <string>
#include <vector>

namespace {

thread_local std::string g_err;

/* ---------------- lattices: Tables 1-3 ---------------- */
struct Lattice {
    int d, Q;
    int c[19][3];
    double w[19];
    int opp[19];
};

/* Table 1, as printed. */
const int D3Q19_C[19][3] = {
    {0, 0, 0},  {+1, 0, 0}, {-1, 0, 0}, {0, +1, 0},  {0, -1, 0},  {0, 0, +1},  {0, 0, -1},
    {+1, +1, 0}, {-1, -1, 0}, {+1, 0, +1}, {-1, 0, -1}, {0, +1, +1}, {0, -1, -1},
    {+1, -1, 0}, {-1, +1, 0}, {+1, 0, -1}, {-1, 0, +1}, {0, +1, -1}, {0, -1, +1}};
/* Table 2; w_4 is printed 1/36, which breaks "weights
 * normalized to unity": c_4=(0,-1) is an axis direction, w_4=1/9 (DESIGN R1). */
const int D2Q9_C[9][3] = {{0, 0, 0},  {+1, 0, 0},  {0, +1, 0},  {-1, 0, 0}, {0, -1, 0},
                          {+1, +1, 0}, {-1, +1, 0}, {-1, -1, 0}, {+1, -1, 0}};
/* Table 3 */
const int D2Q5_C[5][3] = {{0, 0, 0}, {+1, 0, 0}, {0, +1, 0}, {-1, 0, 0}, {0, -1, 0}};
/* D3Q7 is not in the paper; textbook set in the order of D3Q19's first seven (DESIGN R6). */
const int D3Q7_C[7][3] = {{0, 0, 0}, {+1, 0, 0}, {-1, 0, 0}, {0, +1, 0}, {0, -1, 0}, {0, 0, +1}, {0, 0, -1}};

void finish_lattice(Lattice& L) {
    for (int i = 0; i < L.Q; ++i) {
        L.opp[i] = -1;
        for (int j = 0; j < L.Q; ++j)
            if (L.c[j][0] == -L.c[i][0] && L.c[j][1] == -L.c[i][1] && L.c[j][2] == -L.c[i][2]) L.opp[i] = j;
    }
}

Lattice make_flow_lattice(int lattice) {
    Lattice L{};
    if (lattice == REF_D3Q19) {
        L.d = 3; L.Q = 19;
        for (int i = 0; i < 19; ++i) {
            for (int a = 0; a < 3; ++a) L.c[i][a] = D3Q19_C[i][a];
            L.w[i] = (i == 0) ? 1.0 / 3.0 : (i <= 6 ? 1.0 / 18.0 : 1.0 / 36.0);
        }
    } else {
        L.d = 2; L.Q = 9;
        for (int i = 0; i < 9; ++i) {
            for (int a = 0; a < 3; ++a) L.c[i][a] = D2Q9_C[i][a];
            L.w[i] = (i == 0) ? 4.0 / 9.0 : (i <= 4 ? 1.0 / 9.0 : 1.0 / 36.0);
        }
    }
    finish_lattice(L);
    return L;
}

/* scalar lattice: w_0 given (0.4 for D2Q5), the rest share 1-w_0 equally;
 * c_{s,g}^2 = (1-w_0)/d is the only value with sum_i c_i h_i^eq = C u (DESIGN R6). */
Lattice make_scalar_lattice(int lattice, double w0) {
    Lattice L{};
    if (lattice == REF_D3Q19) {
        L.d = 3; L.Q = 7;
        for (int i = 0; i < 7; ++i) for (int a = 0; a < 3; ++a) L.c[i][a] = D3Q7_C[i][a];
    } else {
        L.d = 2; L.Q = 5;
        for (int i = 0; i < 5; ++i) for (int a = 0; a < 3; ++a) L.c[i][a] = D2Q5_C[i][a];
    }
    L.w[0] = w0;
    for (int i = 1; i < L.Q; ++i) L.w[i] = (1.0 - w0) / (double)(L.Q - 1);
    finish_lattice(L);
    return L;
}

/* ---------------- counter-based uniform numbers (DESIGN "Input recipe") ----------------
 * h = splitmix64-finaliser(seed + 0x9E3779B97F4A7C15 * (index + 1)); 53 top bits -> [0,1). */
uint64_t mix64(uint64_t z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
double uniform01(uint64_t seed, uint64_t index) {
    uint64_t h = mix64(seed + 0x9E3779B97F4A7C15ULL * (index + 1ULL));
    return (double)(h >> 11) * (1.0 / 9007199254740992.0);
}

struct Droplet { double cx, cy, cz, r; };

}  // namespace

/* ======================================================================== */
struct ref_ctx {
    int nx, ny, nz, lattice, model, precision;
    virtual ~ref_ctx() {}
    virtual int init(uint64_t seed) = 0;
    virtual int step(int n) = 0;
    virtual int get_macros(void* rho, void* u, void* phi, void* C) = 0;
    virtual int get_force(void* F) = 0;
    virtual int get_populations(void* f) = 0;
    virtual int set_populations(const void* f) = 0;
    virtual size_t population_count() = 0;
    virtual int set_mask(const unsigned char* m) = 0;
};

namespace {

template <class R>
struct Sim : ref_ctx {
    ref_params p;
    Lattice L, Ls;
    int S, d, Q, Qs;
    bool has_sc, has_scalar, has_thermal;
    size_t N;
    bool inited = false;

    /* constants, rounded once to R */
    R w[19], ws[7];
    R omega[2], tau_r[2], omega_c, inv_cs2g;
    R omega_s, inv_rho_solid;      /* solid-phase internal-energy lattice: 1/tau_{e,s} (0: off), 1/rho_s */
    R cfw[2][19];          /* (1 - 1/(2 tau^s)) w_i: prefactor of the Guo term in Eq. 15 */
    R w6[19];              /* 6 w_i = 2 w_i / c_s^2: moving-wall bounce-back (DESIGN R24) */
    R G[2][2], G_ads[2], rho0_psi, force[3], k_react;
    R wall_u[3][2][3];
    R psi_wall;            /* psi(rho_s) of Eq. 12 (single component), 0 when rho_wall = 0 */
    bool moving_walls;
    bool has_walls;

    /* fields */
    std::vector<R> f, fnew;        /* [sigma][i][cell] */
    std::vector<R> h, hnew;        /* [i][cell] */
    std::vector<R> g, gnew;        /* internal-energy lattice [i][cell] (REF_BGK_T), Q directions of the flow lattice */
    std::vector<R> rho, jm, psi;   /* rho[sigma][cell], jm[sigma][a][cell], psi[sigma][cell] */
    std::vector<R> Fv, ub;         /* Fv[sigma][a][cell], ub[a][cell] */
    std::vector<R> ueq;            /* ueq[sigma][a][cell]: equilibrium velocity of the velocity-shift scheme, Eq. 16 */
    std::vector<unsigned char> solid;  /* 1: solid node (bounce-back obstacle), 0: fluid */
    bool has_mask = false;

    R& F_(std::vector<R>& v, int s, int i, size_t cell) { return v[((size_t)s * Q + i) * N + cell]; }
    R& H_(std::vector<R>& v, int i, size_t cell) { return v[(size_t)i * N + cell]; }

    Sim(int nx_, int ny_, int nz_, int lattice_, int model_, const ref_params& pp) : p(pp) {
        nx = nx_; ny = ny_; nz = nz_; lattice = lattice_; model = model_; precision = pp.precision;
        L = make_flow_lattice(lattice);
        double w0s = pp.w0_scalar > 0.0 ? pp.w0_scalar : (lattice == REF_D3Q19 ? 0.25 : 0.4);
        Ls = make_scalar_lattice(lattice, w0s);
        S = (model == REF_SC2 || model == REF_SC2_ADE) ? 2 : 1;
        has_sc = (model == REF_SC1 || model == REF_SC2 || model == REF_SC2_ADE);
        has_walls = pp.bc[0] || pp.bc[1] || pp.bc[2];
        moving_walls = false;
        for (int a = 0; a < 3; ++a)
            for (int sd = 0; sd < 2; ++sd)
                for (int b = 0; b < 3; ++b) {
                    wall_u[a][sd][b] = (R)pp.wall_u[a][sd][b];
                    if (pp.bc[a] == 1 && pp.wall_u[a][sd][b] != 0.0) moving_walls = true;
                }
        has_scalar = (model == REF_SC2_ADE);
        has_thermal = (model == REF_BGK_T);
        d = L.d; Q = L.Q; Qs = Ls.Q;
        N = (size_t)nx * ny * nz;
        for (int i = 0; i < Q; ++i) { w[i] = (R)L.w[i]; w6[i] = (R)(6.0 * L.w[i]); }
        for (int i = 0; i < Qs; ++i) ws[i] = (R)Ls.w[i];
        for (int s = 0; s < 2; ++s) {
            omega[s] = (R)(1.0 / pp.tau[s]);              /* 1/tau, Eq. 15 */
            tau_r[s] = (R)pp.tau[s];
            G_ads[s] = (R)pp.G_ads[s];
            for (int i = 0; i < Q; ++i) cfw[s][i] = (R)((1.0 - 0.5 / pp.tau[s]) * L.w[i]);   /* (1 - 1/(2 tau)) w_i, Eq. 15 */
            for (int t = 0; t < 2; ++t) G[s][t] = (R)pp.G[s][t];
        }
        omega_c = (R)(1.0 / pp.tau_c);                     /* Eq. 34 */
        omega_s = pp.tau_s > 0.0 ? (R)(1.0 / pp.tau_s) : (R)0;     /* Eq. 31 */
        inv_rho_solid = (R)(1.0 / pp.rho_solid);
        inv_cs2g = (R)((double)d / (1.0 - w0s));           /* 1/c_{s,g}^2, Eq. 35, DESIGN R6 */
        rho0_psi = (R)pp.rho0_psi;
        psi_wall = pp.rho_wall > 0.0 ? psi_of((R)pp.rho_wall) : (R)0;
        for (int a = 0; a < 3; ++a) force[a] = (R)pp.force[a];
        k_react = (R)pp.k_react;
        f.assign((size_t)S * Q * N, (R)0); fnew = f;
        if (has_scalar) { h.assign((size_t)Qs * N, (R)0); hnew = h; }
        if (has_thermal) { g.assign((size_t)Q * N, (R)0); gnew = g; }
        rho.assign((size_t)S * N, (R)0);
        jm.assign((size_t)S * 3 * N, (R)0);
        psi.assign((size_t)S * N, (R)0);
        Fv.assign((size_t)S * 3 * N, (R)0);
        ub.assign((size_t)3 * N, (R)0);
        ueq.assign((size_t)S * 3 * N, (R)0);
        solid.assign(N, 0);
    }

    size_t cell_of(int x, int y, int z) const { return (size_t)x + (size_t)nx * ((size_t)y + (size_t)ny * z); }

    /* neighbour x + c; returns false if it lies beyond a wall (bc==1 axis). Periodic axes wrap. */
    bool neighbour(int x, int y, int z, const int* c, size_t& out) const {
        int q[3] = {x + c[0], y + c[1], z + c[2]};
        const int n[3] = {nx, ny, nz};
        for (int a = 0; a < 3; ++a) {
            if (q[a] < 0 || q[a] >= n[a]) {
                if (p.bc[a] == 1) return false;
                q[a] = (q[a] + n[a]) % n[a];
            }
        }
        out = cell_of(q[0], q[1], q[2]);
        return !solid[out];          /* a solid node reflects like a wall */
    }
    /* the same seen from a SOLID node (solid-phase lattice, Eq. 31): its neighbour must be a solid node too; a fluid
     * node or a wall reflects (adiabatic interface: the conjugate coupling Eq. 37-40 is out of scope) */
    bool solid_neighbour(int x, int y, int z, const int* c, size_t& out) const {
        int q[3] = {x + c[0], y + c[1], z + c[2]};
        const int n[3] = {nx, ny, nz};
        for (int a = 0; a < 3; ++a) {
            if (q[a] < 0 || q[a] >= n[a]) {
                if (p.bc[a] == 1) return false;
                q[a] = (q[a] + n[a]) % n[a];
            }
        }
        out = cell_of(q[0], q[1], q[2]);
        return solid[out] != 0;
    }

    /* velocity of the wall a population leaving (x, y, z) along c hits: the first wall axis (x, y, z order) it crosses */
    const R* wall_velocity(int x, int y, int z, const int* c) const {
        const int q[3] = {x + c[0], y + c[1], z + c[2]};
        const int n[3] = {nx, ny, nz};
        for (int a = 0; a < 3; ++a)
            if (p.bc[a] == 1 && (q[a] < 0 || q[a] >= n[a])) return wall_u[a][q[a] < 0 ? 0 : 1];
        return zero3;                /* reflected by a solid node of the mask: at rest */
    }
    R zero3[3] = {(R)0, (R)0, (R)0};

    /* Eq. 10 / Eq. 24, or psi = rho (DESIGN R3) */
    R psi_of(R r) const {
        if (p.psi_kind == 1) return r;
        return rho0_psi * ((R)1 - std::exp(-(r / rho0_psi)));
    }

    /* Eq. 6 with c_s^2 = 1/3: f_i^eq = (w_i rho) e_i, e_i = 1 + 3 cu + 4.5 cu^2 - 1.5 u.u,
     * evaluated as fma(3, cu, fma(4.5 cu, cu, fma(-1.5, u.u, 1))) */
    R eq_poly(int i, const R* u) const {
        R usq = u[0] * u[0];
        for (int a = 1; a < d; ++a) usq = std::fma(u[a], u[a], usq);
        R cu = (R)0;
        for (int a = 0; a < d; ++a) cu = cu + (R)L.c[i][a] * u[a];      /* c = -1, 0, +1: exact products */
        R base = std::fma((R)-1.5, usq, (R)1);
        return std::fma((R)3, cu, std::fma((R)4.5 * cu, cu, base));
    }
    R feq(int i, R rho_s, const R* u) const { return (w[i] * rho_s) * eq_poly(i, u); }

    /* ---- steps 1-4 of one update: moments, psi, force, barycentric velocity ---- */
    void moments_and_force() {
        /* 1. rho^sigma = sum_i f_i, j^sigma = sum_i c_i f_i : Eq. 7-8 / 18 */
        for (int s = 0; s < S; ++s)
            for (size_t cell = 0; cell < N; ++cell) {
                R r = (R)0, j[3] = {(R)0, (R)0, (R)0};
                for (int i = 0; i < Q && !solid[cell]; ++i) {
                    R fi = F_(f, s, i, cell);
                    r = r + fi;
                    for (int a = 0; a < d; ++a) j[a] = j[a] + (R)L.c[i][a] * fi;
                }
                rho[(size_t)s * N + cell] = r;
                for (int a = 0; a < 3; ++a) jm[((size_t)s * 3 + a) * N + cell] = j[a];
            }
        /* 2. pseudopotential of every cell at this time level (full-field barrier; DESIGN R9) */
        for (int s = 0; s < S; ++s)
            for (size_t cell = 0; cell < N; ++cell)
                psi[(size_t)s * N + cell] = solid[cell] ? (R)0 : psi_of(rho[(size_t)s * N + cell]);
        /* 3. Shan-Chen force, Eq. 11 / 13, plus the body force */
        for (int z = 0; z < nz; ++z)
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x) {
                    size_t cell = cell_of(x, y, z);
                    if (solid[cell]) {          /* no fluid here: all fields read as zero */
                        for (int s = 0; s < S; ++s)
                            for (int a = 0; a < 3; ++a) Fv[((size_t)s * 3 + a) * N + cell] = ueq[((size_t)s * 3 + a) * N + cell] = (R)0;
                        for (int a = 0; a < 3; ++a) ub[(size_t)a * N + cell] = (R)0;
                        continue;
                    }
                    R rho_t = rho[cell];
                    for (int s = 1; s < S; ++s) rho_t = rho_t + rho[(size_t)s * N + cell];
                    R inv_rho = (R)1 / rho_t;
                    R acc[2][3] = {{(R)0, (R)0, (R)0}, {(R)0, (R)0, (R)0}};
                    R adh[3] = {(R)0, (R)0, (R)0};   /* sum_i w_i s(x + c_i) c_i over solid neighbours, Eq. 14 */
                    if (has_sc) {
                        for (int t = 0; t < S; ++t)
                            for (int i = 1; i < Q; ++i) {
                                size_t nb;
                                /* Eq. 11 / 12 sum over FLUID neighbours only: a node beyond a wall is solid */
                                if (!neighbour(x, y, z, L.c[i], nb)) continue;
                                for (int a = 0; a < d; ++a)      /* (w_i c_ia) is +-w_i or 0: exact */
                                    acc[t][a] = std::fma(w[i] * (R)L.c[i][a], psi[(size_t)t * N + nb], acc[t][a]);
                            }
                        if (has_walls || has_mask)
                            for (int i = 1; i < Q; ++i) {
                                size_t nb;
                                if (neighbour(x, y, z, L.c[i], nb)) continue;
                                for (int a = 0; a < d; ++a) adh[a] = adh[a] + w[i] * (R)L.c[i][a];
                            }
                    }
                    for (int s = 0; s < S; ++s)
                        for (int a = 0; a < 3; ++a) {
                            /* constant body-force density; split by mass fraction for S=2 (DESIGN R5) */
                            R Fa = (S == 1) ? force[a] : force[a] * (rho[(size_t)s * N + cell] * inv_rho);
                            if (a >= d) Fa = (R)0;
                            if (has_sc && a < d) {
                                /* Eq. 11 / 13: - psi^s(x) sum_t G_st acc^t */
                                R t = G[s][0] * acc[0][a];
                                if (S == 2) t = std::fma(G[s][1], acc[1][a], t);
                                Fa = std::fma(-psi[(size_t)s * N + cell], t, Fa);
                                /* fluid-solid adhesion, Eq. 14: -G_ads rho^s sum_i w_i s c_i */
                                if (has_walls || has_mask) Fa = std::fma(-(G_ads[s] * rho[(size_t)s * N + cell]), adh[a], Fa);
                                /* solid term of Eq. 12, one component: -G psi(x) sum_solid w_i psi(rho_s) c_i */
                                if ((has_walls || has_mask) && S == 1 && p.rho_wall > 0.0)
                                    Fa = std::fma(-(G[0][0] * psi[cell]), psi_wall * adh[a], Fa);
                            }
                            Fv[((size_t)s * 3 + a) * N + cell] = Fa;
                        }
                    /* 4. u^b = (1/rho) sum_sigma [ j^sigma + F^sigma/2 ], Eq. 20-21 */
                    for (int a = 0; a < 3; ++a) {
                        R jt = jm[(size_t)a * N + cell], Ft = Fv[(size_t)a * N + cell];
                        for (int s = 1; s < S; ++s) {
                            jt = jt + jm[((size_t)s * 3 + a) * N + cell];
                            Ft = Ft + Fv[((size_t)s * 3 + a) * N + cell];
                        }
                        ub[(size_t)a * N + cell] = std::fma((R)0.5, Ft, jt) * inv_rho;
                    }
                    /* Shan-Chen (velocity-shift) forcing scheme, p.forcing == 1: common velocity
                     * u' = sum_s (j^s / tau^s) / sum_s (rho^s / tau^s), Eq. 17, and
                     * u^eq,s = u' + tau^s F^s / rho^s, Eq. 16; rho^s u^s = j^s, Eq. 18 */
                    if (p.forcing == 1) {
                        R den = rho[cell] * omega[0];
                        for (int s = 1; s < S; ++s) den = std::fma(rho[(size_t)s * N + cell], omega[s], den);
                        R inv_den = (R)1 / den;
                        for (int a = 0; a < 3; ++a) {
                            R num = jm[(size_t)a * N + cell] * omega[0];
                            for (int s = 1; s < S; ++s) num = std::fma(jm[((size_t)s * 3 + a) * N + cell], omega[s], num);
                            R up = num * inv_den;
                            for (int s = 0; s < S; ++s) {
                                R inv_rs = (R)1 / rho[(size_t)s * N + cell];
                                ueq[((size_t)s * 3 + a) * N + cell] = std::fma(tau_r[s] * Fv[((size_t)s * 3 + a) * N + cell], inv_rs, up);
                            }
                        }
                    }
                }
    }

    /* ---- one time step t -> t+1 ---- */
    void step_once() {
        moments_and_force();
        for (int z = 0; z < nz; ++z)
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x) {
                    size_t cell = cell_of(x, y, z);
                    if (solid[cell]) {          /* solid nodes are not updated: their (unused) populations stay */
                        for (int s = 0; s < S; ++s)
                            for (int i = 0; i < Q; ++i) F_(fnew, s, i, cell) = F_(f, s, i, cell);
                        if (has_scalar) for (int i = 0; i < Qs; ++i) H_(hnew, i, cell) = H_(h, i, cell);
                        if (has_thermal && omega_s > (R)0) {
                            /* solid-phase internal-energy lattice, Eq. 31 with g^eq_{s,i} = w_i rho_s eps_s
                             * (Eq. 32, no velocity) and rho_s eps_s = sum_i g_{s,i} (Eq. 33): pure diffusion with
                             * alpha_s = (tau_{e,s} - 1/2) / 3 among the solid nodes */
                            R E = (R)0;
                            for (int i = 0; i < Q; ++i) E = E + H_(g, i, cell);
                            for (int i = 0; i < Q; ++i) {
                                R gi = H_(g, i, cell);
                                R gstar = std::fma(-omega_s, std::fma(-w[i], E, gi), gi);
                                size_t nb;
                                if (solid_neighbour(x, y, z, L.c[i], nb)) H_(gnew, i, nb) = gstar;
                                else H_(gnew, L.opp[i], cell) = gstar;
                            }
                        } else if (has_thermal) {
                            for (int i = 0; i < Q; ++i) H_(gnew, i, cell) = H_(g, i, cell);
                        }
                        continue;
                    }
                    R u[3] = {ub[cell], ub[N + cell], ub[2 * N + cell]};
                    /* 5. collide each component: Eq. 15 with Eq. 6 and Eq. 22 */
                    for (int s = 0; s < S; ++s) {
                        R Fs[3] = {Fv[((size_t)s * 3 + 0) * N + cell], Fv[((size_t)s * 3 + 1) * N + cell],
                                   Fv[((size_t)s * 3 + 2) * N + cell]};
                        R uF = u[0] * Fs[0];
                        for (int a = 1; a < d; ++a) uF = std::fma(u[a], Fs[a], uF);
                        R m3uF = (R)-3 * uF;
                        R rho_s = rho[(size_t)s * N + cell];
                        /* velocity-shift scheme: equilibrium at u^eq,s, no forcing term F_i */
                        R us[3] = {u[0], u[1], u[2]};
                        if (p.forcing == 1)
                            for (int a = 0; a < 3; ++a) us[a] = ueq[((size_t)s * 3 + a) * N + cell];
                        for (int i = 0; i < Q; ++i) {
                            R fi = F_(f, s, i, cell);
                            /* f_i - f_i^eq with one rounding: f^eq = (w_i rho^s) e_i, Eq. 6 */
                            R dneq = std::fma(-(w[i] * rho_s), eq_poly(i, us), fi);
                            /* f_i - (f_i - f_i^eq)/tau, Eq. 15 */
                            R fstar = std::fma(-omega[s], dneq, fi);
                            if (p.forcing == 0) {
                                R cu = (R)0, cF = (R)0;
                                for (int a = 0; a < d; ++a) cu = cu + (R)L.c[i][a] * u[a];
                                for (int a = 0; a < d; ++a) cF = cF + (R)L.c[i][a] * Fs[a];
                                /* F_i / w_i = 3 (c_i.F - u.F) + 9 (c_i.u)(c_i.F), Eq. 22 with c_s^2 = 1/3 */
                                R Fi = std::fma((R)3, cF, std::fma((R)9 * cu, cF, m3uF));
                                /* + (1 - 1/(2 tau)) F_i, Eq. 15 */
                                fstar = std::fma(cfw[s][i], Fi, fstar);
                            }
                            /* 7. stream, Eq. 5; halfway bounce-back at walls */
                            size_t nb;
                            if (neighbour(x, y, z, L.c[i], nb)) F_(fnew, s, i, nb) = fstar;
                            else {
                                /* moving wall: the reflected population exchanges momentum with the wall,
                                 * f_opp(i)(x, t+1) = f*_i(x, t) - 2 w_i rho (c_i . u_w) / c_s^2 ("Bounce Back
                                 * ... incorporating an additional term"; DESIGN R24), rho the cell's density at t */
                                if (moving_walls) {   /* (mask solids are at rest) */
                                    const R* uw = wall_velocity(x, y, z, L.c[i]);
                                    R cuw = (R)0;
                                    for (int a = 0; a < d; ++a) cuw = cuw + (R)L.c[i][a] * uw[a];
                                    fstar = std::fma(-(w6[i] * rho_s), cuw, fstar);
                                }
                                F_(fnew, s, L.opp[i], cell) = fstar;
                            }
                        }
                    }
                    /* internal-energy lattice (IEDDF), Eq. 27 with g^eq = w_i rho eps [1 + 3 cu + 4.5 cu^2
                     * - 1.5 u.u], Eq. 30 (c_s^2 = 1/3), rho eps = sum_i g_i (Eq. 29); u: DESIGN R25 */
                    if (has_thermal) {
                        R E = (R)0;
                        for (int i = 0; i < Q; ++i) E = E + H_(g, i, cell);
                        for (int i = 0; i < Q; ++i) {
                            R gi = H_(g, i, cell);
                            R gstar = std::fma(-omega_c, std::fma(-(w[i] * E), eq_poly(i, u), gi), gi);
                            size_t nb;
                            if (neighbour(x, y, z, L.c[i], nb)) H_(gnew, i, nb) = gstar;
                            else H_(gnew, L.opp[i], cell) = gstar;     /* adiabatic wall: plain reflection */
                        }
                    }
                    /* 6. scalar lattice: Eq. 34-36 + first-order source (DESIGN R8) */
                    if (has_scalar) {
                        R C = (R)0;
                        for (int i = 0; i < Qs; ++i) C = C + H_(h, i, cell);
                        R rA = rho[cell], rB = rho[N + cell];
                        R inv_rho = (R)1 / (rA + rB);
                        R chi = ((R)4 * (rA * inv_rho)) * (rB * inv_rho);
                        R Rsrc = -((k_react * C) * chi);
                        for (int i = 0; i < Qs; ++i) {
                            R hi = H_(h, i, cell);
                            R cu = (R)0;
                            for (int a = 0; a < d; ++a) cu = cu + (R)Ls.c[i][a] * u[a];
                            /* h_i - h_i^eq, h^eq = (w_i C)(1 + c_i.u / c_sg^2), Eq. 35; relaxation Eq. 34; source w_i R (R8) */
                            R dneq = std::fma(-(ws[i] * C), std::fma(inv_cs2g, cu, (R)1), hi);
                            R hstar = std::fma(ws[i], Rsrc, std::fma(-omega_c, dneq, hi));
                            size_t nb;
                            if (neighbour(x, y, z, Ls.c[i], nb)) H_(hnew, i, nb) = hstar;
                            else H_(hnew, Ls.opp[i], cell) = hstar;
                        }
                    }
                }
        f.swap(fnew);
        if (has_scalar) h.swap(hnew);
        if (has_thermal) g.swap(gnew);
    }

    int step(int n) override {
        if (!inited) { g_err = "ref_step before init / set_populations"; return -4; }
        if (n < 0) { g_err = "n < 0"; return -1; }
        for (int k = 0; k < n; ++k) step_once();
        return 0;
    }

    /* ---- initial macroscopic fields (double), DESIGN "Input recipe" ---- */
    double min_image(double a, double b, int n, int bc) const {
        double dd = std::fabs(a - b);
        if (bc == 0 && (double)n - dd < dd) dd = (double)n - dd;
        return dd;
    }

    std::vector<Droplet> droplet_list(uint64_t seed) const {
        /* sequential draws from stream 2 until the requested volume fraction is reached (DESIGN R18) */
        std::vector<Droplet> v;
        const double PI = 3.14159265358979323846;
        double target = p.vol_frac * (double)N, vol = 0.0;
        uint64_t base = 2ULL * (uint64_t)N;
        for (uint64_t k = 0; vol < target && k < 100000; ++k) {
            Droplet dr;
            dr.cx = (double)nx * uniform01(seed, base + 4 * k + 0);
            dr.cy = (double)ny * uniform01(seed, base + 4 * k + 1);
            dr.cz = (d == 3) ? (double)nz * uniform01(seed, base + 4 * k + 2) : 0.0;
            dr.r = p.rmin + (p.rmax - p.rmin) * uniform01(seed, base + 4 * k + 3);
            vol += (d == 3) ? (4.0 / 3.0) * PI * dr.r * dr.r * dr.r : PI * dr.r * dr.r;
            v.push_back(dr);
        }
        return v;
    }

    int init(uint64_t seed) override {
        const double PI = 3.14159265358979323846;
        std::vector<Droplet> drops;
        if (p.init_kind == REF_INIT_RANDOM_DROPLETS) drops = droplet_list(seed);
        for (int z = 0; z < nz; ++z)
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x) {
                    size_t cell = cell_of(x, y, z);
                    double r0[2] = {p.rho_init[0], p.rho_init[1]};
                    double u0[3] = {0.0, 0.0, 0.0};
                    double c0 = p.c_init;
                    switch (p.init_kind) {
                    case REF_INIT_REST: break;
                    case REF_INIT_TAYLOR_GREEN: {
                        if (d == 2) {
                            /* 2D Taylor-Green vortex (DESIGN R19): the planar analogue of Eq. 45 */
                            double kx = 2.0 * PI / (double)nx, ky = 2.0 * PI / (double)ny;
                            double A = p.u0, B = p.u0 * (kx / ky);
                            u0[0] = -A * std::cos(kx * x) * std::sin(ky * y);
                            u0[1] = B * std::sin(kx * x) * std::cos(ky * y);
                            r0[0] = p.rho_init[0] * (1.0 - 0.75 * (A * A * std::cos(2.0 * kx * x) + B * B * std::cos(2.0 * ky * y)));
                        } else {
                            /* Eq. 45a-c; Eq. 45d is garbled in print, the textbook
                             * P = P0 + rho0 U0^2/16 (cos 2kx + cos 2ky)(cos 2kz + 2) is used (DESIGN R21);
                             * rho = rho0 + 3 (P - P0) */
                            double kx = 2.0 * PI / (double)nx, ky = 2.0 * PI / (double)ny, kz = 2.0 * PI / (double)nz;
                            u0[0] = p.u0 * std::cos(kx * x) * std::sin(ky * y) * std::sin(kz * z);
                            u0[1] = -p.u0 * std::sin(kx * x) * std::cos(ky * y) * std::sin(kz * z);
                            u0[2] = 0.0;
                            r0[0] = p.rho_init[0] * (1.0 + 3.0 * (p.u0 * p.u0 / 16.0) * (std::cos(2.0 * kz * z) + 2.0) *
                                                               (std::cos(2.0 * kx * x) + std::cos(2.0 * ky * y)));
                        }
                        break;
                    }
                    case REF_INIT_DROPLET: {
                        /* tanh profile of width W around a centred droplet (DESIGN R17), then noise */
                        double dx = min_image((double)x, 0.5 * (nx - 1), nx, p.bc[0]);
                        double dy = min_image((double)y, 0.5 * (ny - 1), ny, p.bc[1]);
                        double dz = (d == 3) ? min_image((double)z, 0.5 * (nz - 1), nz, p.bc[2]) : 0.0;
                        double dist = std::sqrt(dx * dx + dy * dy + dz * dz);
                        double th = std::tanh(2.0 * (dist - p.radius) / p.width);
                        double mean = 0.5 * (p.rho_in + p.rho_out), half = 0.5 * (p.rho_in - p.rho_out);
                        r0[0] = mean - half * th;
                        r0[1] = mean + half * th;
                        c0 = p.c_init * (0.5 * (1.0 - th));
                        for (int s = 0; s < S; ++s)
                            r0[s] = r0[s] * (1.0 + p.noise_amp * (2.0 * uniform01(seed, cell + (uint64_t)N * s) - 1.0));
                        break;
                    }
                    case REF_INIT_UNIFORM_NOISE: {
                        for (int s = 0; s < S; ++s)
                            r0[s] = p.rho_init[s] * (1.0 + p.noise_amp * (2.0 * uniform01(seed, cell + (uint64_t)N * s) - 1.0));
                        break;
                    }
                    case REF_INIT_RANDOM_DROPLETS: {
                        /* indicator I = max_k prof((dist_k - r_k)/W), prof = cubic smoothstep (DESIGN R18) */
                        double I = 0.0;
                        for (const Droplet& dr : drops) {
                            double dx = min_image((double)x, dr.cx, nx, p.bc[0]);
                            double dy = min_image((double)y, dr.cy, ny, p.bc[1]);
                            double dz = (d == 3) ? min_image((double)z, dr.cz, nz, p.bc[2]) : 0.0;
                            double s = (std::sqrt(dx * dx + dy * dy + dz * dz) - dr.r) / p.width;
                            double v = (s <= -1.0) ? 1.0 : (s >= 1.0 ? 0.0 : (0.5 - 0.75 * s) + (0.25 * s) * (s * s));
                            if (v > I) I = v;
                        }
                        r0[0] = p.rho_out + (p.rho_in - p.rho_out) * I;
                        r0[1] = p.rho_in - (p.rho_in - p.rho_out) * I;
                        c0 = p.c_init * I;
                        break;
                    }
                    default: g_err = "bad init_kind"; return -1;
                    }
                    /* populations = equilibrium at (rho, u), no non-equilibrium part (DESIGN R10) */
                    R u[3] = {(R)u0[0], (R)u0[1], (R)u0[2]};
                    for (int s = 0; s < S; ++s)
                        for (int i = 0; i < Q; ++i) F_(f, s, i, cell) = feq(i, (R)r0[s], u);
                    if (has_scalar)
                        for (int i = 0; i < Qs; ++i) {
                            R cu = (R)0;
                            for (int a = 0; a < d; ++a) cu = cu + (R)Ls.c[i][a] * u[a];
                            H_(h, i, cell) = (ws[i] * (R)c0) * std::fma(inv_cs2g, cu, (R)1);
                        }
                    if (has_thermal)      /* g_i = g^eq(rho eps, u), eps = c_init */
                        for (int i = 0; i < Q; ++i) H_(g, i, cell) = feq(i, (R)r0[0] * (R)c0, u);
                }
        inited = true;
        return 0;
    }

    int get_macros(void* rho_o, void* u_o, void* phi_o, void* C_o) override {
        if (!inited) { g_err = "get_macros before init"; return -4; }
        if (C_o && !has_scalar && !has_thermal) { g_err = "model has no scalar lattice"; return -1; }
        moments_and_force();
        if (rho_o) std::memcpy(rho_o, rho.data(), sizeof(R) * S * N);
        if (u_o) std::memcpy(u_o, ub.data(), sizeof(R) * d * N);
        if (phi_o) {
            R* ph = (R*)phi_o;
            for (size_t cell = 0; cell < N; ++cell) {
                if (solid[cell]) { ph[cell] = (R)0; continue; }
                if (S == 2) {
                    R rA = rho[cell], rB = rho[N + cell];
                    R inv_rho = (R)1 / (rA + rB);
                    ph[cell] = (rA - rB) * inv_rho;
                } else {
                    ph[cell] = psi[cell];
                }
            }
        }
        if (C_o) {
            R* Cc = (R*)C_o;
            for (size_t cell = 0; cell < N; ++cell) {
                R C = (R)0;
                if (has_thermal) {      /* internal energy eps = sum_i g_i / rho, Eq. 29 */
                    if (!solid[cell]) {
                        for (int i = 0; i < Q; ++i) C = C + H_(g, i, cell);
                        C = C * ((R)1 / rho[cell]);
                    } else if (omega_s > (R)0) {   /* eps_s = sum_i g_{s,i} / rho_s, Eq. 33 */
                        for (int i = 0; i < Q; ++i) C = C + H_(g, i, cell);
                        C = C * inv_rho_solid;
                    }
                    Cc[cell] = C;
                    continue;
                }
                for (int i = 0; i < Qs && !solid[cell]; ++i) C = C + H_(h, i, cell);
                Cc[cell] = C;
            }
        }
        return 0;
    }

    int get_force(void* F) override {
        if (!inited) { g_err = "get_force before init"; return -4; }
        moments_and_force();
        R* o = (R*)F;
        for (int s = 0; s < S; ++s)
            for (int a = 0; a < d; ++a)
                std::memcpy(o + ((size_t)s * d + a) * N, &Fv[((size_t)s * 3 + a) * N], sizeof(R) * N);
        return 0;
    }

    int set_mask(const unsigned char* m) override {
        has_mask = false;
        for (size_t cell = 0; cell < N; ++cell) {
            solid[cell] = m ? (m[cell] != 0) : 0;
            if (solid[cell]) has_mask = true;
        }
        return 0;
    }

    size_t population_count() override { return (size_t)S * Q * N + (has_scalar ? (size_t)Qs * N : 0) + (has_thermal ? (size_t)Q * N : 0); }

    int get_populations(void* out) override {
        if (!inited) { g_err = "get_populations before init"; return -4; }
        R* o = (R*)out;
        std::memcpy(o, f.data(), sizeof(R) * f.size());
        if (has_scalar) std::memcpy(o + f.size(), h.data(), sizeof(R) * h.size());
        if (has_thermal) std::memcpy(o + f.size(), g.data(), sizeof(R) * g.size());
        return 0;
    }
    int set_populations(const void* in) override {
        const R* o = (const R*)in;
        std::memcpy(f.data(), o, sizeof(R) * f.size());
        if (has_scalar) std::memcpy(h.data(), o + f.size(), sizeof(R) * h.size());
        if (has_thermal) std::memcpy(g.data(), o + f.size(), sizeof(R) * g.size());
        inited = true;
        return 0;
    }
};

}  // namespace

extern "C" {

ref_ctx* ref_create(int nx, int ny, int nz, int lattice, int model, const ref_params* p) {
    if (!p || p->struct_size != sizeof(ref_params)) { g_err = "bad params / struct_size"; return nullptr; }
    if (nx < 1 || ny < 1 || nz < 1) { g_err = "bad grid"; return nullptr; }
    if (lattice != REF_D2Q9 && lattice != REF_D3Q19) { g_err = "bad lattice"; return nullptr; }
    if (lattice == REF_D2Q9 && nz != 1) { g_err = "D2Q9 needs nz == 1"; return nullptr; }
    if (model < REF_BGK || model > REF_BGK_T) { g_err = "bad model"; return nullptr; }
    if (p->precision != 32 && p->precision != 64) { g_err = "precision must be 32 or 64"; return nullptr; }
    if (p->forcing != 0 && p->forcing != 1) { g_err = "forcing must be 0 (Guo) or 1 (velocity shift)"; return nullptr; }
    if (p->psi_kind != 0 && p->psi_kind != 1) { g_err = "bad psi_kind"; return nullptr; }
    int S = (model == REF_SC2 || model == REF_SC2_ADE) ? 2 : 1;
    for (int s = 0; s < S; ++s)
        if (!(p->tau[s] > 0.5)) { g_err = "tau must exceed 0.5"; return nullptr; }
    if ((model == REF_SC2_ADE || model == REF_BGK_T) && !(p->tau_c > 0.5)) { g_err = "tau_c must exceed 0.5"; return nullptr; }
    if (p->tau_s != 0.0 && (model != REF_BGK_T || !(p->tau_s > 0.5) || !(p->rho_solid > 0.0))) {
        g_err = "tau_s (solid-phase lattice) needs REF_BGK_T, tau_s > 0.5 and rho_solid > 0";
        return nullptr;
    }
    for (int a = 0; a < 3; ++a) {
        if (p->bc[a] != 0 && p->bc[a] != 1) { g_err = "bad bc"; return nullptr; }

    }
    if (lattice == REF_D2Q9 && p->bc[2] != 0) { g_err = "2D: bc[2] must be 0"; return nullptr; }
    if (model != REF_BGK && p->psi_kind == 0 && !(p->rho0_psi > 0.0)) { g_err = "rho0_psi must be > 0"; return nullptr; }
    try {
        if (p->precision == 64) return new Sim<double>(nx, ny, nz, lattice, model, *p);
        return new Sim<float>(nx, ny, nz, lattice, model, *p);
    } catch (const std::bad_alloc&) {
        g_err = "out of memory";
        return nullptr;
    }
}

int ref_init_from_seed(ref_ctx* c, uint64_t seed) { return c ? c->init(seed) : -1; }
int ref_step(ref_ctx* c, int n) { return c ? c->step(n) : -1; }
int ref_get_macros(ref_ctx* c, void* rho, void* u, void* phi, void* C) { return c ? c->get_macros(rho, u, phi, C) : -1; }
int ref_get_force(ref_ctx* c, void* F) { return c ? c->get_force(F) : -1; }
int ref_set_mask(ref_ctx* c, const unsigned char* mask) { return c ? c->set_mask(mask) : -1; }
int ref_get_populations(ref_ctx* c, void* f) { return c ? c->get_populations(f) : -1; }
int ref_set_populations(ref_ctx* c, const void* f) { return c ? c->set_populations(f) : -1; }
size_t ref_population_count(ref_ctx* c) { return c ? c->population_count() : 0; }
void ref_destroy(ref_ctx* c) { delete c; }
const char* ref_last_error(void) { return g_err.c_str(); }

/* lattice tables as the oracle uses them, for the golden-table test:
 * kind 0 = flow lattice, 1 = scalar lattice (default w0).  c is Q*3 ints, w is Q doubles. */
int ref_lattice_table(int lattice, int kind, int* Q, int* c, double* w) {
    Lattice L = kind == 0 ? make_flow_lattice(lattice) : make_scalar_lattice(lattice, lattice == REF_D3Q19 ? 0.25 : 0.4);
    *Q = L.Q;
    for (int i = 0; i < L.Q; ++i) {
        for (int a = 0; a < 3; ++a) c[3 * i + a] = L.c[i][a];
        w[i] = L.w[i];
    }
    return 0;
}

}  // extern "C"
