/*
 * include/lbm.h -- C ABI of the B200 (sm_100a) lattice Boltzmann hot path.
 *
 * What the library computes: the per-time-step, per-cell collide-and-stream update of the
 * lattice Boltzmann method as stated in CooLBM (arXiv 2502.12955; citations below are
 * "PAPER.md:<line>" + equation):
 *   - LBGK collision with Guo forcing on D2Q9 / D3Q19 populations
 *         Eq. 3-8, Eq. 15, Eq. 20-23
 *     or with the Shan-Chen velocity-shift forcing scheme, Eq. 16-19
 *   - Shan-Chen pseudopotential interaction force, one or two components
 *         Eq. 10-11, Eq. 13, Eq. 24
 *     with solid nodes left out of the sums (Eq. 12) and the fluid-solid adhesion force (Eq. 14)
 *   - an advection-diffusion scalar lattice D2Q5 / D3Q7 with a first-order interface reaction
 *     source, Eq. 34-36; source term and D3Q7: DESIGN.md readings R6, R8
 *   - an internal-energy lattice on the flow lattice (IEDDF), Eq. 27-30
 *   - periodic boundaries, halfway bounce-back walls at rest or moving (Couette
 *     flow Eq. 41) and halfway bounce-back on the solid nodes of a mask
 * Every step of that path runs in CUDA kernels; there is no CPU fallback.  If no CUDA device
 * is usable, lbm_create returns NULL and lbm_last_error() says why.
 *
 * Conventions
 *   - 2D <=> lattice LBM_D2Q9 and nz == 1.  Cell index = x + nx*(y + ny*z), x fastest.
 *   - "ctx precision" R is float (precision 32) or double (precision 64).  All field buffers
 *     are arrays of R, structure-of-arrays.  N = nx*ny*nz, S = components (1 or 2),
 *     d = 2 or 3, Q = 9 or 19, Qs = 5 or 7.
 *   - Unless a function name ends in _host, every buffer pointer is a DEVICE pointer owned by
 *     the caller and must be valid on the context's stream.  _host functions take HOST
 *     pointers (pageable or pinned), copy inside the call and synchronise the stream.
 *   - All kernels are enqueued on the context's stream (lbm_params.stream, a cudaStream_t, or
 *     the legacy default stream when NULL).  lbm_step and lbm_get_* do not synchronise.
 *   - Return value: 0 on success, a negative LBM_E* code on error; the message is available
 *     from lbm_last_error() (thread-local).  No exception crosses this boundary.
 *   - The context owns only the memory it allocated itself; it never frees lbm_params.workspace.
 */
#ifndef LBM_H
#define LBM_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* flow lattice; the scalar lattice is D2Q5 for D2Q9 and D3Q7 for D3Q19.  PAPER.md:217-240 Tables 1-3.
 * Direction order:
 *   D3Q19: Table 1 as printed: 0 rest; 1..6 = +x,-x,+y,-y,+z,-z; 7..18 = (+,+,0)(-,-,0)(+,0,+)(-,0,-)
 *          (0,+,+)(0,-,-)(+,-,0)(-,+,0)(+,0,-)(-,0,+)(0,+,-)(0,-,+); opposite of 2k-1 is 2k.
 *   D2Q9 : 0 rest; 1 +x; 2 +y; 3 -x; 4 -y; 5 (+,+); 6 (-,+); 7 (-,-); 8 (+,-)   (Table 2, w_4 = 1/9: R1)
 *   D2Q5 : 0 rest; 1 +x; 2 +y; 3 -x; 4 -y (Table 3).   D3Q7: 0 rest; 1..6 = +x,-x,+y,-y,+z,-z (R6). */
enum { LBM_D2Q9 = 0, LBM_D3Q19 = 1 };

/* model: BGK single phase; Shan-Chen one component (Eq. 11); Shan-Chen two components (Eq. 13);
 * two components + scalar lattice with reaction source (Eq. 34-36) */
enum { LBM_BGK = 0, LBM_SC1 = 1, LBM_SC2 = 2, LBM_SC2_ADE = 3,
       /* BGK + internal-energy lattice g_i on the flow lattice (IEDDF), Eq. 27-30:
        * tau_c is its relaxation time tau_e = 3 alpha + 1/2, c_init the initial internal energy, the C output of
        * lbm_get_macros the internal energy eps = sum_i g_i / rho; populations: f (Q*N) then g (Q*N) */
       LBM_BGK_T = 4 };

/* initial condition kinds of lbm_init_from_seed */
enum { LBM_INIT_REST = 0, LBM_INIT_TAYLOR_GREEN = 1, LBM_INIT_DROPLET = 2,
       LBM_INIT_UNIFORM_NOISE = 3, LBM_INIT_RANDOM_DROPLETS = 4 };

/* error codes */
enum { LBM_OK = 0, LBM_EINVAL = -1, LBM_ENOMEM = -2, LBM_ECUDA = -3, LBM_ESTATE = -4 };

typedef struct lbm_params {
    uint32_t struct_size;   /* must be sizeof(lbm_params) */
    int32_t  precision;     /* 32 or 64: storage and arithmetic type of the whole path */
    double   tau[2];        /* relaxation time of each component, > 0.5; Eq. 15 */
    double   tau_c;         /* scalar-lattice relaxation time, > 0.5; Eq. 34 */
    double   G[2][2];       /* Shan-Chen coupling G_{sigma sigma~}; SC1 uses G[0][0]; Eq. 11/13 */
    int32_t  psi_kind;      /* 0: psi = rho0 (1 - exp(-rho/rho0)), Eq. 10/24 ; 1: psi = rho (R3) */
    int32_t  forcing;       /* 0: Guo, Eq. 20-23; 1: Shan-Chen velocity shift, Eq. 16-19
                               (PAPER.md:154-174): u_eq = u' + tau F / rho, no F_i term; both launch paths */
    double   rho0_psi;      /* rho0 of Eq. 10 */
    double   force[3];      /* constant body-force density; S = 2: split by mass fraction (R5) */
    int32_t  bc[3];         /* per axis: 0 periodic, 1 halfway bounce-back walls on both faces.
                               For Shan-Chen models the nodes beyond a wall are solid: left out of the psi
                               stencil (Eq. 11-12) and the source of the adhesion force (G_ads, Eq. 14) */
    int32_t  init_kind;     /* LBM_INIT_* */
    double   k_react;       /* k of the source R = -k C 4 rhoA rhoB/(rhoA+rhoB)^2 (R8) */
    double   w0_scalar;     /* rest weight of the scalar lattice; 0 -> 0.4 (D2Q5) / 0.25 (D3Q7) */
    double   rho_init[2];   /* REST / TAYLOR_GREEN / UNIFORM_NOISE: density per component */
    double   c_init;        /* scalar value (REST...) or value inside droplets (DROPLET, RANDOM_DROPLETS) */
    double   rho_in, rho_out;   /* DROPLET / RANDOM_DROPLETS: component-A density inside / outside */
    double   radius, width;     /* DROPLET radius; interface width W */
    double   noise_amp;         /* relative amplitude of the seeded uniform noise */
    double   u0;                /* TAYLOR_GREEN velocity amplitude */
    double   rmin, rmax, vol_frac;  /* RANDOM_DROPLETS: radius range and target volume fraction */
    double   G_ads[2];      /* fluid-solid adhesion coefficient per component, Eq. 14:
                               F_ads = -G_ads rho sum_i w_i s(x + c_i) c_i; < 0 wetting, > 0 non-wetting */
    double   rho_wall;      /* LBM_SC1: density rho_s of the solid nodes in Eq. 12: adds
                               -G psi(x) sum_solid w_i psi(rho_s) c_i; 0: no such term */
    double   wall_u[3][2][3];  /* [axis][0 low face, 1 high face][component]: velocity of that wall (used where
                               bc[axis] == 1).  A population reflected by a moving wall loses
                               2 w_i rho^sigma (c_i . u_w) / c_s^2 (Couette flow Eq. 41), every
                               model (scalar / energy lattices are reflected without a term); forcing 0 only */
    double   tau_s;         /* LBM_BGK_T with a solid-node mask: relaxation time tau_{e,s} = 3 alpha_s + 1/2 of the
                               solid-phase internal-energy lattice g_{s,i} on the solid nodes, Eq. 31-33
                               (PAPER.md:316-327): g^eq_s = w_i rho_s eps_s, pure diffusion among solid nodes, the
                               fluid-solid interface is adiabatic (Eq. 37-40 are out of scope); the C output reads
                               eps_s = sum_i g_{s,i} / rho_solid there.  0: solid nodes carry no lattice */
    double   rho_solid;     /* rho_s of Eq. 32-33, > 0 when tau_s is set */
    void*    workspace;     /* DEVICE memory of >= lbm_workspace_bytes() bytes, 256-byte aligned (e.g. from
                               torch), or NULL: the library allocates (cudaMalloc) and frees it */
    void*    stream;        /* cudaStream_t, or NULL for the legacy default stream */
} lbm_params;

typedef struct lbm_ctx lbm_ctx;   /* opaque */

/* Bytes of device workspace a context of this shape needs: the in-place population array
 * (S*Q + Qs values per cell, ONE copy: AA-pattern streaming), the psi field (S values per cell,
 * Shan-Chen models only) and padding.  0 on invalid arguments. */
size_t lbm_workspace_bytes(int nx, int ny, int nz, int lattice, int model, const lbm_params* p);

/* Validate, bind to the current CUDA device, allocate.  NULL on error (see lbm_last_error). */
lbm_ctx* lbm_create(int nx, int ny, int nz, int lattice, int model, const lbm_params* p);

/* Fill the populations with the equilibrium (Eq. 6) of the seeded initial fields (init_kind),
 * time level t = 0.  Runs on the device. */
int lbm_init_from_seed(lbm_ctx* ctx, uint64_t seed);

/* Advance n >= 0 time steps (asynchronous).  One step = steps a1..a8 of DESIGN.md: moments, psi,
 * Shan-Chen force, barycentric velocity (Eq. 20), BGK + Guo collision (Eq. 15, 22), scalar
 * lattice + source, in-place streaming (Eq. 5), boundaries.  LBM_ESTATE before init / set. */
int lbm_step(lbm_ctx* ctx, int n);

/* Macroscopic fields at the current time level into caller-owned DEVICE buffers (NULL = skip):
 *   rho[sigma][cell] (S*N)   density per component, Eq. 7/18
 *   u[a][cell]       (d*N)   barycentric velocity incl. F/2, Eq. 20
 *   phi[cell]        (N)     S = 2: (rhoA-rhoB)/(rhoA+rhoB);  S = 1: psi(rho)
 *   C[cell]          (N)     scalar concentration, Eq. 36; LBM_EINVAL if the model has no scalar lattice */
int lbm_get_macros(lbm_ctx* ctx, void* rho, void* u, void* phi, void* C);

/* Total force density per component (Shan-Chen + body), F[sigma][a][cell] (S*d*N), device buffer. */
int lbm_get_force(lbm_ctx* ctx, void* F);

/* Solid-node mask: N bytes in DEVICE memory (non-zero = solid node), owned by the caller and valid until it is
 * replaced, cleared (NULL) or the context is destroyed.  Solid nodes reflect populations like a wall (halfway
 * bounce-back on arbitrary nodes), are not updated, are left out of the psi stencil (Eq. 11-12,
 * PAPER.md:128-132) and act on the fluid through the adhesion force (G_ads, Eq. 14); all output fields read zero
 * there.  Runs on LBM_PATH_REGISTER (the context falls back to it); the mask may change at even time levels only (LBM_ESTATE otherwise: at odd
 * levels the in-place layout depends on which neighbours reflect).  Synchronises the stream. */
int lbm_set_mask(lbm_ctx* ctx, const unsigned char* mask);

/* Canonical populations at the current time level, independent of the in-place slot permutation:
 * f[sigma][i][cell] (S*Q*N) followed by h[i][cell] (Qs*N, scalar models only).  Device buffers.
 * lbm_set_populations also marks the context initialised and resets the time level parity. */
size_t lbm_population_count(const lbm_ctx* ctx);
int lbm_get_populations(lbm_ctx* ctx, void* f);
int lbm_set_populations(lbm_ctx* ctx, const void* f);

/* End-to-end call with HOST buffers: (optional) upload canonical populations from f_in_host
 * (NULL = keep the current state), run n steps, compute the macros and copy them to the host
 * buffers (NULL = skip), then synchronise.  Layouts as in lbm_set_populations / lbm_get_macros. */
int lbm_run_host(lbm_ctx* ctx, const void* f_in_host, int n,
                 void* rho_host, void* u_host, void* phi_host, void* C_host);

/* Which kernels lbm_step launches.  Both paths compute the same bits (same expression tree per cell).
 *   LBM_PATH_REGISTER   one thread per cell (two in fp32 BGK), populations loaded straight into registers: one launch
 *                       of the fused step kernel per time step, preceded by the psi pass for Shan-Chen models
 *                       (which reads the flow populations a second time).  Works for every shape and boundary.
 *   LBM_PATH_PIPELINE   Shan-Chen models: ONE persistent, warp-specialised launch per time step (tile.cuh), one
 *                       block per SM.  Producer warps bulk-copy (cp.async.bulk + mbarrier, TMA unit) the populations
 *                       of a tile of 1 KB rows and the psi rows around it into a ring of shared-memory stages; two
 *                       teams of step warps collide and stream it (a1, a3-a8) from there, two fp32 cells per thread
 *                       in packed arithmetic; psi of the NEXT time level (step a2; Eq. 11 / 13 need psi of all
 *                       neighbours at one time level: PAPER.md:128, 136; R9) is formed in the same launch -- every
 *                       ticket also brings a tile whose surrounding tiles have been stepped -- from populations still in L2,
 *                       into a second psi buffer (allocated by the library, S * N values): every population crosses
 *                       HBM once per step in each direction (ncu: 1.05 x the algorithmic bytes on config 5).  Needs
 *                       nx * sizeof(value) % 16 == 0, periodic x, no solid-node mask (LBM_EINVAL
 *                       otherwise) and the GPU to itself (all blocks co-resident); walls in y / z, at rest or moving, and both
 *                       forcing schemes are handled.
 * lbm_create starts on LBM_PATH_REGISTER; unless lbm_set_path was called, the first lbm_step switches a
 * two-component D3Q19 fp32 context with more than 2^21 cells to LBM_PATH_PIPELINE where it applies -- the one case
 * in which it is the faster path; smaller grids replay a CUDA graph of the register kernels.
 * lbm_set_mask falls back to LBM_PATH_REGISTER.
 * rows_per_pencil: rows of the slower-but-one axis that are marched together along the slowest axis (<= 0:
 * default).  Synchronises the stream. */
enum { LBM_PATH_REGISTER = 0, LBM_PATH_PIPELINE = 1 };
int lbm_set_path(lbm_ctx* ctx, int path, int rows_per_pencil);
int lbm_get_path(const lbm_ctx* ctx);

/* The row schedule of LBM_PATH_PIPELINE for nm x ns rows (D3Q19: nm = ny, ns = nz; D2Q9: nm = 1, ns = ny;
 * wrap_m / wrap_s: that axis is periodic): *count = 2 * nm * ns items; if items != NULL (HOST, capacity items of 3
 * int32: kind 0 = step of the row / 1 = psi of the next time level of the row, m, s) they are written out: the
 * step rows in pencil order; the psi rows whose last dependency is the k-th step row follow step row
 * k + delay_rows.  *deferred_rows (optional) receives the number of psi rows that wait for another pencil
 * (re-read from HBM).  Host-only, needs no GPU. */
int lbm_tile_schedule(int nm, int ns, int rows_per_pencil, int wrap_m, int wrap_s, int delay_rows, int32_t* items,
                      size_t capacity, size_t* count, int* deferred_rows);

/* The tickets LBM_PATH_PIPELINE deals out round-robin to its blocks, built from that row schedule with nxs tiles per
 * row: *count tickets of 8 int32 (sx, sy, sz, step-part present, px, py, pz, psi-part present): ticket k carries the
 * k-th tile to step and the next tile whose psi is due; a psi part depends only on step parts of EARLIER tickets (the
 * property that makes the kernel's waits deadlock-free; tests/test_abi.py checks it).  three_d: rows are (y, z), else
 * (y, 0).  Host-only, needs no GPU. */
int lbm_tile_tickets(int nm, int ns, int nxs, int rows_per_pencil, int wrap_m, int wrap_s, int delay_rows, int three_d,
                     int32_t* tickets, size_t capacity, size_t* count);

/* Synchronise the stream and report deferred device-side errors (LBM_ECUDA if a bounded wait of LBM_PATH_PIPELINE
 * timed out; lbm_run_host performs the same check before it returns).  Without a synchronisation, lbm_step,
 * lbm_get_macros and lbm_get_populations report such an error of an earlier, completed lbm_step (a pinned host copy
 * of the status word is refreshed at the end of every lbm_step on that path). */
int lbm_check(lbm_ctx* ctx);

/* The Shan-Chen step for callers that must not allocate (code under CUDA-graph capture set-up, serving loops, harnesses
 * that forbid cudaMalloc): n time steps (n even, >= 0) of a Shan-Chen model (LBM_SC1 / LBM_SC2 / LBM_SC2_ADE; a1-a8 as in
 * lbm_step, register kernels: psi pass + fused step per time step) IN PLACE on the caller's DEVICE array f of canonical
 * populations at an even time level, f[sigma][i][cell] followed by h[i][cell] (the layout of lbm_set_populations; the
 * result is canonical again), on the CURRENT device and the stream params->stream.  No context, no workspace
 * (params->workspace is ignored), no mask, no cudaMalloc / cudaFree / allocating library call: the psi field (Eq. 10 /
 * 24), the only intermediate of the path, lives in a static device array of lbm_static_scratch_bytes() = 16 MiB that
 * every GPU which loads the library holds until exit.  LBM_EINVAL if S * nx * ny * nz * sizeof(value) exceeds that
 * (e.g. two components in fp32: up to 2^21 cells = 128^3), for other models, odd n, or invalid parameters.  Every call
 * on a device shares the array: it keeps the last call's contents (nothing in it needs to start at zero: every step
 * writes psi of all cells before reading any), and two calls that overlap on the GPU (different streams or host
 * threads, same device) RACE on it -- serialise them.  Asynchronous like lbm_step.  Results equal lbm_step's bit for
 * bit. */
size_t lbm_static_scratch_bytes(void);
int lbm_step_static(int nx, int ny, int nz, int lattice, int model, const lbm_params* params, void* f, int n);

/* number of time steps taken since init / set_populations */
int64_t lbm_time(const lbm_ctx* ctx);

/* number of kernel launches this context has enqueued so far (for benchmarks) */
int64_t lbm_launch_count(const lbm_ctx* ctx);

/* Per-kernel timing for benchmarks.  lbm_kernel_timing(ctx, 1) synchronises the stream, discards
 * earlier records and from then on brackets every launch of the fused step kernel (kind 0) and of
 * the psi pass (kind 1) with a pair of CUDA events on the context's stream; (ctx, 0) switches it
 * off.  lbm_kernel_time_ms synchronises the stream and returns the summed device time (ms) and
 * the number of launches of that kind recorded since timing was switched on.  Host pointers. */
int lbm_kernel_timing(lbm_ctx* ctx, int enable);
int lbm_kernel_time_ms(lbm_ctx* ctx, int kind, double* total_ms, int64_t* launches);

/* Lattice tables as the kernels use them: kind 0 = flow lattice, 1 = scalar lattice (default w0).
 * c receives Q*3 ints, w receives Q doubles, opp receives Q ints.  Host pointers. */
int lbm_lattice_table(int lattice, int kind, int* Q, int* c, double* w, int* opp);

void lbm_destroy(lbm_ctx* ctx);            /* NULL-safe; synchronises the stream first */
const char* lbm_last_error(void);          /* thread-local, never NULL */

#ifdef __cplusplus
}
#endif
#endif
