/*
 * oracle/ref_lbm.h -- C ABI of the CPU ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, single-threaded CPU implementation of the lattice Boltzmann
 * update of CooLBM (arXiv 2502.12955).  It exists only so that tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * can check and time the CUDA library against it.  It shares no code with
 * paper_2502_12955_b200/ and nothing in the product path may call it.
 *
 * All pointers are HOST pointers.  Field outputs are in the context precision
 * (float for precision==32, double for precision==64), structure-of-arrays,
 * cell index = x + nx*(y + ny*z).
 *
 * Citations are PAPER.md line numbers + equation.
 */
#ifndef REF_LBM_H
#define REF_LBM_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* flow lattice (scalar lattice is D2Q5 / D3Q7 respectively); Tables 1-3 */
enum { REF_D2Q9 = 0, REF_D3Q19 = 1 };
/* model: BGK (Eq. 3-8), single-component Shan-Chen (Eq. 11), two-component Shan-Chen (Eq. 13),
 * two-component Shan-Chen + advection-diffusion scalar lattice (Eq. 34-36) with reaction source */
enum { REF_BGK = 0, REF_SC1 = 1, REF_SC2 = 2, REF_SC2_ADE = 3,
       REF_BGK_T = 4 /* BGK + internal-energy lattice g_i on the flow lattice, Eq. 27-30 */ };
/* init kinds */
enum { REF_INIT_REST = 0, REF_INIT_TAYLOR_GREEN = 1, REF_INIT_DROPLET = 2,
       REF_INIT_UNIFORM_NOISE = 3, REF_INIT_RANDOM_DROPLETS = 4 };

typedef struct ref_params {
    uint32_t struct_size;   /* = sizeof(ref_params) */
    int32_t  precision;     /* 32 or 64 */
    double   tau[2];        /* flow relaxation time per component, Eq. 15 */
    double   tau_c;         /* scalar relaxation time, Eq. 34 */
    double   G[2][2];       /* Shan-Chen coupling G_{sigma sigma~}, Eq. 11/13 */
    int32_t  psi_kind;      /* 0: rho0*(1-exp(-rho/rho0)) Eq. 10/24 ; 1: psi = rho */
    int32_t  forcing;       /* 0: Guo, Eq. 20-23; 1: Shan-Chen velocity shift, Eq. 16-19 */
    double   rho0_psi;      /* rho0 of Eq. 10 */
    double   force[3];      /* constant body-force density */
    int32_t  bc[3];         /* per axis: 0 periodic, 1 halfway bounce-back walls */
    int32_t  init_kind;
    double   k_react;       /* first-order reaction rate of the scalar source */
    double   w0_scalar;     /* rest weight of the scalar lattice; 0 -> 0.4 (D2Q5) / 0.25 (D3Q7) */
    double   rho_init[2];
    double   c_init;
    double   rho_in, rho_out, radius, width, noise_amp, u0, rmin, rmax, vol_frac;
    double   G_ads[2];      /* fluid-solid adhesion coefficient per component, Eq. 14; solid = beyond a wall */
    double   rho_wall;      /* SC1: density rho_s of the solid nodes in Eq. 12; 0: no such term */
    double   wall_u[3][2][3]; /* velocity of the wall at the low / high face of each wall axis (moving-wall bounce-back) */
    double   tau_s;         /* REF_BGK_T: relaxation time tau_{e,s} = 3 alpha_s + 1/2 of the solid-phase internal-energy lattice g_{s,i} on
                             * the solid nodes of the mask, Eq. 31-33; 0: solid nodes carry no lattice */
    double   rho_solid;     /* rho_s of Eq. 32-33 (eps_s = sum_i g_{s,i} / rho_s) */
} ref_params;

typedef struct ref_ctx ref_ctx;

ref_ctx* ref_create(int nx, int ny, int nz, int lattice, int model, const ref_params* p); /* NULL on error */
int  ref_init_from_seed(ref_ctx*, uint64_t seed);
int  ref_step(ref_ctx*, int n);
/* rho: S*N, u: d*N, phi: N, C: N ; any pointer may be NULL */
int  ref_get_macros(ref_ctx*, void* rho, void* u, void* phi, void* C);
/* total force density per component (Shan-Chen + body), F[sigma][a][cell], S*d*N */
int  ref_get_force(ref_ctx*, void* F);
/* solid-node mask, N bytes (non-zero = solid), NULL clears it: solid nodes reflect populations like a wall
 * (halfway bounce-back), are left out of the psi stencil (Eq. 11-12) and act in Eq. 14 */
int  ref_set_mask(ref_ctx*, const unsigned char* mask);
/* canonical populations f[sigma][i][cell] (S*Q*N) then h[i][cell] (Qs*N, scalar models only) */
int  ref_get_populations(ref_ctx*, void* f);
int  ref_set_populations(ref_ctx*, const void* f);
size_t ref_population_count(ref_ctx*);   /* number of values get/set_populations moves */
void ref_destroy(ref_ctx*);
const char* ref_last_error(void);
/* lattice tables as the oracle uses them (kind 0: flow lattice, 1: scalar lattice with default w0);
 * c receives Q*3 ints, w receives Q doubles */
int  ref_lattice_table(int lattice, int kind, int* Q, int* c, double* w);

#ifdef __cplusplus
}
#endif
#endif
