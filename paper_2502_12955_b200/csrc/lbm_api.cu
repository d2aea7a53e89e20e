// C ABI of the B200 lattice Boltzmann library (include/lbm.h): context, validation, launch logic.
// All compute runs in the kernels of kernels.cuh; there is no CPU path.
#include "../../include/lbm.h"

#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "dispatch.h"
#include "kernels.cuh"
#include "tile.cuh"

namespace {

// rows per pencil of the resident-tile schedule unless the caller chooses (lbm_set_path)
#ifndef LBM_TILE_DEFAULT_PY
#define LBM_TILE_DEFAULT_PY 32
#endif
// rounds of the round-robin between a STEP ticket and the PSI tickets that depend on it (tile_schedule.h)
#ifndef LBM_TILE_DELAY
#define LBM_TILE_DELAY 7
#endif

thread_local std::string g_err;
#ifdef LBM_TILE_TRACE
long long* g_trace = nullptr;
#endif

int fail(int code, const std::string& msg) {
    g_err = msg;
    return code;
}
int cuda_fail(cudaError_t e, const char* what) {
    g_err = std::string(what) + ": " + cudaGetErrorString(e);
    return LBM_ECUDA;
}
#define CK(call)                                              \
    do {                                                      \
        cudaError_t e_ = (call);                              \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);   \
    } while (0)

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Shape {
    int S, Q, Qs, d;
    bool sc, scalar;
    size_t N, B;
    size_t f_bytes, h_bytes, psi_bytes, total;
};

// returns empty string if valid
std::string validate(int nx, int ny, int nz, int lattice, int model, const lbm_params* p, Shape* sh) {
    if (!p) return "params is NULL";
    if (p->struct_size != sizeof(lbm_params)) return "params.struct_size != sizeof(lbm_params)";
    if (nx < 1 || ny < 1 || nz < 1) return "grid extents must be >= 1";
    if (lattice != LBM_D2Q9 && lattice != LBM_D3Q19) return "unknown lattice";
    if (lattice == LBM_D2Q9 && nz != 1) return "D2Q9 needs nz == 1";
    if (model < LBM_BGK || model > LBM_BGK_T) return "unknown model";
    if (p->precision != 32 && p->precision != 64) return "precision must be 32 or 64";
    if (p->forcing != 0 && p->forcing != 1) return "forcing must be 0 (Guo) or 1 (Shan-Chen velocity shift)";
    if (p->psi_kind != 0 && p->psi_kind != 1) return "psi_kind must be 0 or 1";
    if ((double)nx * (double)ny * (double)nz > 2147483647.0) return "grid has more than 2^31-1 cells";
    if (ny > 65535 || nz > 65535) return "ny and nz must not exceed 65535 (CUDA grid limits)";
    if ((lattice == LBM_D3Q19 ? 19.0 : 9.0) * (double)nx * (double)ny * (double)nz >= 4294967296.0)
        return "Q * nx * ny * nz must stay below 2^32 (the kernels index one lattice with 32 bits)";
    const int S = (model == LBM_SC2 || model == LBM_SC2_ADE) ? 2 : 1;
    for (int s = 0; s < S; ++s)
        if (!(p->tau[s] > 0.5)) return "tau must exceed 0.5";
    if ((model == LBM_SC2_ADE || model == LBM_BGK_T) && !(p->tau_c > 0.5)) return "tau_c must exceed 0.5";
    if (model == LBM_BGK_T && p->forcing != 0) return "LBM_BGK_T runs with Guo forcing only";
    for (int a = 0; a < 3; ++a) {
        if (p->bc[a] != 0 && p->bc[a] != 1) return "bc must be 0 (periodic) or 1 (bounce-back walls)";
    }
    if (lattice == LBM_D2Q9 && p->bc[2] != 0) return "2D: bc[2] must be 0";
    if (model != LBM_BGK && p->psi_kind == 0 && !(p->rho0_psi > 0.0)) return "rho0_psi must be > 0";
    if (p->w0_scalar < 0.0 || p->w0_scalar >= 1.0) return "w0_scalar must lie in [0, 1)";
    if (p->rho_wall < 0.0) return "rho_wall must be >= 0";
    if (p->tau_s != 0.0 && (model != LBM_BGK_T || !(p->tau_s > 0.5) || !(p->rho_solid > 0.0)))
        return "tau_s (solid-phase lattice) needs LBM_BGK_T, tau_s > 0.5 and rho_solid > 0";
    if (p->init_kind < LBM_INIT_REST || p->init_kind > LBM_INIT_RANDOM_DROPLETS) return "unknown init_kind";
    for (int a = 0; a < 3; ++a)
        for (int sd = 0; sd < 2; ++sd)
            for (int b = 0; b < 3; ++b)
                if (p->bc[a] == 1 && p->wall_u[a][sd][b] != 0.0 && p->forcing != 0)
                    return "moving walls (wall_u) are implemented for Guo forcing (forcing = 0) only";
    if (sh) {
        sh->S = S;
        sh->d = lattice == LBM_D3Q19 ? 3 : 2;
        sh->Q = lattice == LBM_D3Q19 ? 19 : 9;
        sh->Qs = lattice == LBM_D3Q19 ? 7 : 5;
        if (model == LBM_BGK_T) sh->Qs = sh->Q;            // second lattice = internal-energy lattice on the flow lattice
        sh->sc = model == LBM_SC1 || model == LBM_SC2 || model == LBM_SC2_ADE;
        sh->scalar = model == LBM_SC2_ADE || model == LBM_BGK_T;     // has a second lattice (KP::h) of Qs values per cell
        sh->N = (size_t)nx * ny * nz;
        sh->B = p->precision == 64 ? 8 : 4;
        sh->f_bytes = align_up((size_t)S * sh->Q * sh->N * sh->B, 256);
        sh->h_bytes = sh->scalar ? align_up((size_t)sh->Qs * sh->N * sh->B, 256) : 0;
        sh->psi_bytes = sh->sc ? align_up((size_t)S * sh->N * sh->B, 256) : 0;
        sh->total = sh->f_bytes + sh->h_bytes + sh->psi_bytes;
    }
    return "";
}

struct DeviceGuard {
    int prev = -1;
    bool changed = false;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) changed = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() { if (changed) cudaSetDevice(prev); }
};

}  // namespace

struct lbm_ctx {
    int nx, ny, nz, lattice, model;
    lbm_params p;
    Shape sh;
    int device;
    cudaStream_t stream;
    char* ws;
    bool owns_ws;
    void *f, *h, *psi;
    const lbm::Ops* ops;
    lbm::KP<double> kp64;
    lbm::KP<float> kp32;
    bool walls;
    bool moving;          // some wall has a velocity (moving-wall bounce-back)
    bool bc_walls;        // walls from lbm_params.bc (walls = bc_walls || a mask is set)
    int forced;           // 0 no force, 1 Guo forcing, 2 velocity-shift forcing (kernel variant)
    bool inited;
    int64_t t;
    int64_t launches;
    double4* droplets_dev;
    void* scratch;        // device staging for lbm_run_host outputs
    size_t scratch_bytes;
    // per-kernel timing (lbm_kernel_timing): event pairs around every launch of kind 0 (fused step) / 1 (psi pass)
    bool timing;
    std::vector<cudaEvent_t> ev[2];
    int path;                         // LBM_PATH_*: which kernels lbm_step launches
    // small grids (launch-latency bound): GRAPH_STEPS time steps of the register path captured once as a CUDA
    // graph and replayed, so that consecutive kernels start back to back instead of one launch call each
    cudaGraphExec_t graph_exec;
    cudaStream_t graph_capture_stream;
    bool graph_failed;
    // resident-tile path (tile.cuh): schedule, flags, second psi buffer
    int tile_py;                      // rows per pencil in use
    int tile_blocks;                  // blocks per launch
    lbm::TileItem* tile_items;        // device copy of the schedule: the STEP tickets, then the PSI tickets
    long long tile_n_items;           // tiles = STEP tickets = PSI tickets
    void* psi_ws;                     // the psi buffer inside the workspace
    void* psi_alt;                    // the psi buffer the resident-tile kernel writes psi(t + 1) to (swapped with psi after every launch)
    int64_t psi_t;                    // time level of the values in psi (-1: none)
    int tile_nxs;
    int* tile_flags;                  // one int per tile, then the status word
    size_t tile_n_tiles;
    int tile_epoch;
    bool path_user_set;               // the caller chose the path (lbm_set_path): no automatic switch
    int* tile_status_host;            // pinned host mirror of the device status word, refreshed after every lbm_step on the tile path

    const void* kp() const { return p.precision == 64 ? (const void*)&kp64 : (const void*)&kp32; }
    // kernel variant: 0 fully periodic, 1 bounce-back walls (bc), 2 with a solid-node mask
    int wmode() const { return kp64.mask ? 2 : (bc_walls ? 1 : 0); }
};

namespace {

template <class R>
void fill_kp(lbm::KP<R>& k, const lbm_ctx* c) {
    const lbm_params& p = c->p;
    k.f = (R*)c->f; k.h = (R*)c->h; k.psi = (R*)c->psi;
    k.nx = c->nx; k.ny = c->ny; k.nz = c->nz; k.N = (int)c->sh.N;
    for (int a = 0; a < 3; ++a) { k.bc[a] = p.bc[a]; k.force[a] = (R)p.force[a]; }
    k.psi_kind = p.psi_kind;
    // constants are formed in double and rounded once to R
    for (int s = 0; s < 2; ++s) {
        k.omega[s] = (R)(1.0 / p.tau[s]);
        // (1 - 1/(2 tau)) w per weight class (rest, axis, diagonal), formed in double from the double weights
        const double wc[3] = {c->lattice == LBM_D3Q19 ? lbm::D3Q19::w(0) : lbm::D2Q9::w(0),
                              c->lattice == LBM_D3Q19 ? lbm::D3Q19::w(1) : lbm::D2Q9::w(1),
                              c->lattice == LBM_D3Q19 ? lbm::D3Q19::w(18) : lbm::D2Q9::w(8)};
        for (int kc = 0; kc < 3; ++kc) k.cfw[s][kc] = (R)((1.0 - 0.5 / p.tau[s]) * wc[kc]);
        k.tau[s] = (R)p.tau[s];
        for (int t = 0; t < 2; ++t) k.G[s][t] = (R)p.G[s][t];
        k.G_ads[s] = (R)p.G_ads[s];
    }
    const double w0s = p.w0_scalar > 0.0 ? p.w0_scalar : (c->lattice == LBM_D3Q19 ? 0.25 : 0.4);
    k.omega_c = (R)(1.0 / p.tau_c);
    k.inv_cs2g = (R)((double)c->sh.d / (1.0 - w0s));
    k.ws0 = (R)w0s;
    k.ws1 = (R)((1.0 - w0s) / (double)((c->lattice == LBM_D3Q19 ? 7 : 5) - 1));
    for (int a = 0; a < 3; ++a)
        for (int sd = 0; sd < 2; ++sd)
            for (int b = 0; b < 3; ++b) k.wall_u[a][sd][b] = (R)p.wall_u[a][sd][b];
    k.mask = nullptr;
    k.solid_term = p.rho_wall > 0.0 ? 1 : 0;
    {   // psi(rho_s) in the context precision, the same expression as psi_of in the kernels
        const R rw = (R)p.rho_wall, r0 = (R)p.rho0_psi;
        k.psi_wall = p.rho_wall > 0.0 ? (p.psi_kind == 1 ? rw : r0 * ((R)1 - std::exp(-(rw / r0)))) : (R)0;
    }
    k.rho0_psi = (R)p.rho0_psi;
    k.k_react = (R)p.k_react;
    k.omega_s = p.tau_s > 0.0 ? (R)(1.0 / p.tau_s) : (R)0;
    k.inv_rho_solid = p.tau_s > 0.0 ? (R)(1.0 / p.rho_solid) : (R)0;
}

// host copy of the counter-based generator (integer arithmetic, bit-identical to the device one)
uint64_t h_mix64(uint64_t z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
double h_uniform01(uint64_t seed, uint64_t index) {
    return (double)(h_mix64(seed + 0x9E3779B97F4A7C15ULL * (index + 1ULL)) >> 11) * (1.0 / 9007199254740992.0);
}

// RANDOM_DROPLETS (R18): sequential draws (cx, cy, cz, r) from stream 2 until the volume fraction is reached
std::vector<double4> droplet_list(const lbm_ctx* c, uint64_t seed) {
    std::vector<double4> v;
    const double PI = 3.14159265358979323846;
    const double N = (double)c->sh.N;
    const double target = c->p.vol_frac * N;
    double vol = 0.0;
    const uint64_t base = 2ULL * (uint64_t)c->sh.N;
    for (uint64_t k = 0; vol < target && k < 100000; ++k) {
        double4 dr;
        dr.x = (double)c->nx * h_uniform01(seed, base + 4 * k + 0);
        dr.y = (double)c->ny * h_uniform01(seed, base + 4 * k + 1);
        dr.z = (c->sh.d == 3) ? (double)c->nz * h_uniform01(seed, base + 4 * k + 2) : 0.0;
        dr.w = c->p.rmin + (c->p.rmax - c->p.rmin) * h_uniform01(seed, base + 4 * k + 3);
        vol += (c->sh.d == 3) ? (4.0 / 3.0) * PI * dr.w * dr.w * dr.w : PI * dr.w * dr.w;
        v.push_back(dr);
    }
    return v;
}

// event before / after a launch of the given kind while kernel timing is on
int mark(lbm_ctx* c, int kind) {
    if (!c->timing) return 0;
    cudaEvent_t e;
    CK(cudaEventCreate(&e));
    c->ev[kind].push_back(e);
    CK(cudaEventRecord(e, c->stream));
    return 0;
}

void drop_events(lbm_ctx* c) {
    for (int k = 0; k < 2; ++k) {
        for (cudaEvent_t e : c->ev[k]) cudaEventDestroy(e);
        c->ev[k].clear();
    }
}

int run_psi(lbm_ctx* c) {
    int rc = mark(c, 1);
    if (rc) return rc;
    CK(c->ops->psi(c->kp(), c->model, (int)(c->t & 1), c->wmode(), c->stream));
    c->launches++;
    c->psi_t = c->t;
    return mark(c, 1);
}

void set_psi(lbm_ctx* c, void* psi) {
    c->psi = psi;
    c->kp64.psi = (double*)psi;
    c->kp32.psi = (float*)psi;
}

void tile_free(lbm_ctx* c) {
    if (c->tile_items) cudaFree(c->tile_items);
    if (c->tile_flags) cudaFree(c->tile_flags);
    if (c->psi_alt) {
        // psi and psi_alt swap after every launch: free whichever of the two is not the workspace buffer
        void* extra = c->psi == c->psi_ws ? c->psi_alt : c->psi;
        if (c->psi != c->psi_ws) { set_psi(c, c->psi_ws); c->psi_t = -1; }
        cudaFree(extra);
    }
    if (c->tile_status_host) cudaFreeHost(c->tile_status_host);
    c->tile_items = nullptr; c->tile_flags = nullptr; c->psi_alt = nullptr; c->tile_status_host = nullptr;
    c->path = LBM_PATH_REGISTER;
}

// what the resident-tile kernel handles (tile.cuh): Shan-Chen models with either forcing scheme, periodic x, 16-byte aligned
// rows, walls in y / z at rest, no solid-node mask
const char* tile_ineligible(const lbm_ctx* c) {
    if (!c->sh.sc) return "LBM_PATH_PIPELINE exists for the Shan-Chen models (BGK already moves the algorithmic bytes)";
    if (c->kp64.mask) return "a solid-node mask runs on LBM_PATH_REGISTER only";
    if (c->p.bc[0] != 0) return "LBM_PATH_PIPELINE needs periodic x";
    if (((size_t)c->nx * c->sh.B) % 16 != 0) return "LBM_PATH_PIPELINE needs nx * sizeof(value) to be a multiple of 16 bytes";
    return nullptr;
}

// Switch to the resident-tile path: build the schedule (one STEP and one PSI ticket per tile), the flags and the
// second psi buffer; py <= 0 picks the default
int path_setup(lbm_ctx* c, int py) {
    CK(cudaStreamSynchronize(c->stream));
    tile_free(c);
    const Shape& sh = c->sh;
    const int nm = sh.d == 3 ? c->ny : 1, ns = sh.d == 3 ? c->nz : c->ny;
    const bool wrap_m = sh.d == 3 ? c->p.bc[1] == 0 : true, wrap_s = sh.d == 3 ? c->p.bc[2] == 0 : c->p.bc[1] == 0;
    const int tx = c->ops->tile_tx();
    const int nxs = (c->nx + tx - 1) / tx;
    const int walls = c->bc_walls ? 1 : 0;
    const int vshift = c->forced == 2 ? 1 : 0;
    int resident = c->ops->tile_blocks(c->model, 0, walls, vshift);
    const int r1 = c->ops->tile_blocks(c->model, 1, walls, vshift);
    if (r1 < resident) resident = r1;
    if (resident < 1) return fail(LBM_ECUDA, "resident-tile kernel: occupancy query failed");
    // default pencil: one plane of the pencil (what the psi pass trails the step by) stays far below the L2 capacity
    if (py <= 0) py = LBM_TILE_DEFAULT_PY;
    if (py < 1) py = 1;
    if (py > nm) py = nm;
    const size_t n_tiles = (size_t)nm * ns * nxs;
    if ((double)n_tiles > 1.0e9) return fail(LBM_EINVAL, "resident-tile path: more than 1e9 tiles");
    const int blocks = (long long)resident < (long long)n_tiles ? resident : (int)n_tiles;
    // a PSI ticket comes LBM_TILE_DELAY rounds of the round-robin after the last STEP ticket it depends on
    int delay_tiles = LBM_TILE_DELAY * blocks;
#ifdef LBM_TUNING
    if (const char* e = getenv("LBM_TILE_DELAY")) delay_tiles = atoi(e);
#endif
    const int delay_rows = (delay_tiles + nxs - 1) / nxs;
    const std::vector<lbm::TileRow> rows = lbm::tile_schedule(nm, ns, py, wrap_m, wrap_s, delay_rows, nullptr);
    const std::vector<lbm::TileItem> items = lbm::tile_tickets(rows, nxs, sh.d == 3);
    if (items.size() < n_tiles) return fail(LBM_ECUDA, "resident-tile path: inconsistent schedule");
    c->tile_py = py;
    c->tile_blocks = blocks;
    c->tile_n_items = (long long)items.size();
    c->tile_nxs = nxs;
    c->tile_n_tiles = n_tiles;
    cudaError_t e = cudaMalloc((void**)&c->tile_items, items.size() * sizeof(lbm::TileItem));
    if (e == cudaSuccess) e = cudaMalloc((void**)&c->tile_flags, (c->tile_n_tiles + 1) * sizeof(int));    // flags, status word
    if (e == cudaSuccess) e = cudaMalloc(&c->psi_alt, sh.psi_bytes);
    if (e == cudaSuccess) e = cudaHostAlloc((void**)&c->tile_status_host, sizeof(int), cudaHostAllocDefault);
    if (e == cudaSuccess) *c->tile_status_host = 0;
    if (e != cudaSuccess) { cudaGetLastError(); tile_free(c); return fail(LBM_ENOMEM, "cudaMalloc of the schedule failed"); }
    CK(cudaMemcpyAsync(c->tile_items, items.data(), items.size() * sizeof(lbm::TileItem), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemsetAsync(c->tile_flags, 0, (c->tile_n_tiles + 1) * sizeof(int), c->stream));
    CK(cudaStreamSynchronize(c->stream));   // items goes out of scope
    c->tile_epoch = 0;
    c->path = LBM_PATH_PIPELINE;
    return 0;
}

int run_tile(lbm_ctx* c) {
    const int parity = (int)(c->t & 1);
    if (c->psi_t != c->t) {              // first step on this path (or after new populations): psi(t) by the psi pass
        int rc = run_psi(c);
        if (rc) return rc;
    }
    if (c->tile_epoch == 0x7fffffff) {   // epoch wrap: clear the flags (once per 2^31 - 1 launches)
        CK(cudaMemsetAsync(c->tile_flags, 0, c->tile_n_tiles * sizeof(int), c->stream));
        c->tile_epoch = 0;
    }
    lbm::TileArgs wa;
    wa.items = c->tile_items;
    wa.n_items = (unsigned)c->tile_n_items;
    wa.nxs = c->tile_nxs;
    wa.flags = c->tile_flags;
    wa.epoch = ++c->tile_epoch;
    wa.status = c->tile_flags + c->tile_n_tiles;
    wa.psi_out = c->psi_alt;
    wa.moving = c->moving ? 1 : 0;
#ifdef LBM_TILE_TRACE
    if (!g_trace) { cudaMalloc((void**)&g_trace, sizeof(long long) * 10 * 4096); cudaMemset(g_trace, 0, sizeof(long long) * 10 * 4096); }
    wa.trace = g_trace;
#endif
    int rc = mark(c, 0);
    if (rc) return rc;
    CK(c->ops->tile(c->kp(), c->model, parity, c->bc_walls ? 1 : 0, c->forced == 2 ? 1 : 0, &wa, c->tile_blocks, c->stream));
    c->launches++;
    // the launch has written psi(t + 1) to psi_alt: it is the current buffer from now on
    void* cur = c->psi;
    set_psi(c, c->psi_alt);
    c->psi_alt = cur;
    c->psi_t = c->t + 1;
    return mark(c, 0);
}

// The status word as of the last lbm_step that has COMPLETED on the tile path (its copy into the pinned mirror is the
// last thing that call enqueues): a timed-out wait is reported by the next API call at the latest, without a
// synchronisation; lbm_check / lbm_run_host report it exactly
int tile_status_seen(lbm_ctx* c) {
    if (c->tile_status_host && *(volatile int*)c->tile_status_host != 0)
        return fail(LBM_ECUDA, "resident-tile kernel: a bounded wait timed out in an earlier lbm_step (status " +
                                   std::to_string(*(volatile int*)c->tile_status_host) + "); the state is invalid");
    return 0;
}

// deferred device-side error of the resident-tile path (a bounded wait gave up); the stream must be idle
int tile_status(lbm_ctx* c) {
    if (c->path == LBM_PATH_REGISTER) return 0;
    int st = 0;
    CK(cudaMemcpy(&st, c->tile_flags + c->tile_n_tiles, sizeof(int), cudaMemcpyDeviceToHost));
    if (st != 0)
        return fail(LBM_ECUDA, "resident-tile kernel: a bounded wait timed out (bits: 1 stage load, 2 free stage, 4 publisher, 8 flags of the "
                               "tiles around a psi tile): " + std::to_string(st) + "; the state is invalid");
    return 0;
}

int ensure_scratch(lbm_ctx* c, size_t bytes) {
    if (c->scratch_bytes >= bytes) return 0;
    if (c->scratch) { cudaFree(c->scratch); c->scratch = nullptr; c->scratch_bytes = 0; }
    cudaError_t e = cudaMalloc(&c->scratch, bytes);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(LBM_ENOMEM, "cudaMalloc of the host-transfer staging buffer failed"); }
    c->scratch_bytes = bytes;
    return 0;
}

}  // namespace

extern "C" {

const char* lbm_last_error(void) { return g_err.c_str(); }

size_t lbm_workspace_bytes(int nx, int ny, int nz, int lattice, int model, const lbm_params* p) {
    Shape sh;
    std::string e = validate(nx, ny, nz, lattice, model, p, &sh);
    if (!e.empty()) { g_err = e; return 0; }
    return sh.total;
}

lbm_ctx* lbm_create(int nx, int ny, int nz, int lattice, int model, const lbm_params* p) {
    Shape sh;
    std::string e = validate(nx, ny, nz, lattice, model, p, &sh);
    if (!e.empty()) { g_err = "lbm_create: " + e; return nullptr; }
    int ndev = 0;
    cudaError_t ce = cudaGetDeviceCount(&ndev);
    if (ce != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        g_err = std::string("lbm_create: no usable CUDA device (") + (ce != cudaSuccess ? cudaGetErrorString(ce) : "device count 0") +
                "); this library has no CPU path";
        return nullptr;
    }
    lbm_ctx* c = new (std::nothrow) lbm_ctx();
    if (!c) { g_err = "lbm_create: out of host memory"; return nullptr; }
    c->nx = nx; c->ny = ny; c->nz = nz; c->lattice = lattice; c->model = model;
    c->p = *p; c->sh = sh;
    c->stream = (cudaStream_t)p->stream;
    c->inited = false; c->t = 0; c->launches = 0;
    c->droplets_dev = nullptr; c->scratch = nullptr; c->scratch_bytes = 0;
    c->timing = false;
    c->graph_exec = nullptr; c->graph_capture_stream = nullptr; c->graph_failed = false;
    c->path = LBM_PATH_REGISTER; c->tile_items = nullptr; c->tile_flags = nullptr;
    c->tile_py = 0; c->tile_blocks = 0; c->tile_epoch = 0; c->path_user_set = false; c->tile_status_host = nullptr;
    if (cudaGetDevice(&c->device) != cudaSuccess) { g_err = "lbm_create: cudaGetDevice failed"; delete c; return nullptr; }
    if (p->workspace) {
        if (((uintptr_t)p->workspace & 255u) != 0) { g_err = "lbm_create: workspace must be 256-byte aligned"; delete c; return nullptr; }
        c->ws = (char*)p->workspace; c->owns_ws = false;
    } else {
        void* w = nullptr;
        ce = cudaMalloc(&w, sh.total);
        if (ce != cudaSuccess) {
            cudaGetLastError();
            g_err = std::string("lbm_create: cudaMalloc of the workspace failed: ") + cudaGetErrorString(ce);
            delete c;
            return nullptr;
        }
        c->ws = (char*)w; c->owns_ws = true;
    }
    c->f = c->ws;
    c->h = sh.scalar ? c->ws + sh.f_bytes : nullptr;
    c->psi = sh.sc ? c->ws + sh.f_bytes + sh.h_bytes : nullptr;
    c->psi_ws = c->psi; c->psi_alt = nullptr; c->psi_t = -1;
    c->bc_walls = p->bc[0] || p->bc[1] || p->bc[2];
    c->walls = c->bc_walls;
    c->moving = false;
    for (int a = 0; a < 3; ++a)
        for (int sd = 0; sd < 2; ++sd)
            for (int b = 0; b < 3; ++b)
                if (p->bc[a] == 1 && p->wall_u[a][sd][b] != 0.0) c->moving = true;
    c->forced = (sh.sc || p->force[0] != 0.0 || p->force[1] != 0.0 || p->force[2] != 0.0) ? 1 : 0;
    if (p->forcing == 1) c->forced = 2;       // its own arithmetic even when the force is zero
    if (p->precision == 64) c->ops = lattice == LBM_D3Q19 ? lbm::ops_f64_d3q19() : lbm::ops_f64_d2q9();
    else c->ops = lattice == LBM_D3Q19 ? lbm::ops_f32_d3q19() : lbm::ops_f32_d2q9();
    fill_kp(c->kp64, c);
    fill_kp(c->kp32, c);
    return c;
}

void lbm_destroy(lbm_ctx* c) {
    if (!c) return;
    DeviceGuard g(c->device);
    cudaStreamSynchronize(c->stream);
    drop_events(c);
    if (c->droplets_dev) cudaFree(c->droplets_dev);
    if (c->scratch) cudaFree(c->scratch);
    tile_free(c);
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    if (c->graph_capture_stream) cudaStreamDestroy(c->graph_capture_stream);
    if (c->owns_ws && c->ws) cudaFree(c->ws);
    cudaGetLastError();
    delete c;
}

int lbm_init_from_seed(lbm_ctx* c, uint64_t seed) {
    if (!c) return fail(LBM_EINVAL, "ctx is NULL");
    DeviceGuard g(c->device);
    lbm::InitArgs ia;
    std::memset(&ia, 0, sizeof(ia));
    ia.kind = c->p.init_kind; ia.seed = seed;
    ia.rho_init[0] = c->p.rho_init[0]; ia.rho_init[1] = c->p.rho_init[1];
    ia.c_init = c->p.c_init; ia.rho_in = c->p.rho_in; ia.rho_out = c->p.rho_out;
    ia.radius = c->p.radius; ia.width = c->p.width; ia.noise_amp = c->p.noise_amp; ia.u0 = c->p.u0;
    ia.droplets = nullptr; ia.n_droplets = 0;
    if (c->p.init_kind == LBM_INIT_RANDOM_DROPLETS) {
        std::vector<double4> v = droplet_list(c, seed);
        if (c->droplets_dev) { cudaStreamSynchronize(c->stream); cudaFree(c->droplets_dev); c->droplets_dev = nullptr; }
        if (!v.empty()) {
            CK(cudaMalloc((void**)&c->droplets_dev, v.size() * sizeof(double4)));
            CK(cudaMemcpyAsync(c->droplets_dev, v.data(), v.size() * sizeof(double4), cudaMemcpyHostToDevice, c->stream));
            CK(cudaStreamSynchronize(c->stream));   // v goes out of scope
        }
        ia.droplets = c->droplets_dev; ia.n_droplets = (int)v.size();
    }
    CK(c->ops->init(c->kp(), c->model, &ia, c->stream));
    c->launches++;
    c->inited = true;
    c->t = 0;
    c->psi_t = -1;
    return 0;
}

namespace {
constexpr int GRAPH_STEPS = 32;                 // even: a replay starts and ends at even parity
constexpr size_t GRAPH_MAX_CELLS = 1u << 21;    // above this a step takes far longer than a launch call

// Default launch path, chosen at the first step unless the caller chose one (lbm_set_path): the resident-tile kernel
// where it applies AND is the faster of the two (measured): the two-component D3Q19 models in fp32 on
// grids too large for the CUDA-graph replay.  (D2Q9 in fp64: the register kernels are faster.)
void choose_default_path(lbm_ctx* c) {
    if (c->path_user_set || c->path != LBM_PATH_REGISTER) return;
    c->path_user_set = true;                    // decide once
    if (c->sh.N <= GRAPH_MAX_CELLS || tile_ineligible(c) != nullptr) return;
    if (!(c->lattice == LBM_D3Q19 && c->p.precision == 32 && c->sh.S == 2)) return;
    if (path_setup(c, 0) != 0) { cudaGetLastError(); tile_free(c); }
}

// the kernels of one time step of the register path, enqueued on st (no event marks, no counters)
int enqueue_register_step(lbm_ctx* c, int parity, cudaStream_t st) {
    if (c->sh.sc) CK(c->ops->psi(c->kp(), c->model, parity, c->wmode(), st));
    CK(c->ops->step(c->kp(), c->model, parity, c->wmode(), c->forced, c->moving ? 1 : 0, st));
    return 0;
}

// capture GRAPH_STEPS steps on a private stream (nothing runs during capture) and instantiate the graph
int build_graph(lbm_ctx* c) {
    cudaGraph_t graph = nullptr;
    if (!c->graph_capture_stream) CK(cudaStreamCreateWithFlags(&c->graph_capture_stream, cudaStreamNonBlocking));
    CK(cudaStreamBeginCapture(c->graph_capture_stream, cudaStreamCaptureModeRelaxed));
    int rc = 0;
    for (int k = 0; k < GRAPH_STEPS && rc == 0; ++k) rc = enqueue_register_step(c, k & 1, c->graph_capture_stream);
    cudaError_t e = cudaStreamEndCapture(c->graph_capture_stream, &graph);
    if (rc != 0 || e != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        return rc != 0 ? rc : fail(LBM_ECUDA, "CUDA graph capture failed");
    }
    e = cudaGraphInstantiate(&c->graph_exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) { cudaGetLastError(); c->graph_exec = nullptr; return cuda_fail(e, "cudaGraphInstantiate"); }
    return 0;
}
}  // namespace

int lbm_step(lbm_ctx* c, int n) {
    if (!c) return fail(LBM_EINVAL, "ctx is NULL");
    if (!c->inited) return fail(LBM_ESTATE, "lbm_step before lbm_init_from_seed / lbm_set_populations");
    if (n < 0) return fail(LBM_EINVAL, "n < 0");
    DeviceGuard g(c->device);
    { int rs = tile_status_seen(c); if (rs) return rs; }
    if ((c->t & 1) == 0) choose_default_path(c);
    int done = 0;
    if (c->path == LBM_PATH_REGISTER && !c->timing && !c->graph_failed && c->sh.N <= GRAPH_MAX_CELLS) {
        if ((c->t & 1) && n >= GRAPH_STEPS + 1) {       // reach even parity with one ordinary step
            int rc = enqueue_register_step(c, 1, c->stream);
            if (rc) return rc;
            c->launches += c->sh.sc ? 2 : 1; c->t++; done++;
        }
        if ((c->t & 1) == 0 && n - done >= GRAPH_STEPS) {
            if (!c->graph_exec && build_graph(c) != 0) c->graph_failed = true;    // fall back to plain launches
            while (c->graph_exec && n - done >= GRAPH_STEPS) {
                CK(cudaGraphLaunch(c->graph_exec, c->stream));
                c->launches += (int64_t)GRAPH_STEPS * (c->sh.sc ? 2 : 1);
                c->t += GRAPH_STEPS; done += GRAPH_STEPS;
            }
        }
    }
    for (int k = done; k < n; ++k) {
        const int parity = (int)(c->t & 1);
        int rc;
        if (c->path != LBM_PATH_REGISTER) {   // one persistent launch per step (tile.cuh)
            if ((rc = run_tile(c))) return rc;
            c->t++;
            continue;
        }
        if (c->sh.sc) {   // a2: psi of every cell at this time level (full-field barrier, R9)
            rc = run_psi(c);
            if (rc) return rc;
        }
        if ((rc = mark(c, 0))) return rc;
        CK(c->ops->step(c->kp(), c->model, parity, c->wmode(), c->forced, c->moving ? 1 : 0, c->stream));
        c->launches++;
        if ((rc = mark(c, 0))) return rc;
        c->t++;
    }
    if (c->path != LBM_PATH_REGISTER && n > done)
        CK(cudaMemcpyAsync(c->tile_status_host, c->tile_flags + c->tile_n_tiles, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    return 0;
}

int lbm_get_macros(lbm_ctx* c, void* rho, void* u, void* phi, void* C) {
    if (!c) return fail(LBM_EINVAL, "ctx is NULL");
    if (!c->inited) return fail(LBM_ESTATE, "lbm_get_macros before init");
    if (C && !c->sh.scalar) return fail(LBM_EINVAL, "model has no scalar lattice");
    DeviceGuard g(c->device);
    { int rs = tile_status_seen(c); if (rs) return rs; }
    if (c->sh.sc && c->psi_t != c->t) { int rc = run_psi(c); if (rc) return rc; }
    CK(c->ops->macros(c->kp(), c->model, (int)(c->t & 1), c->wmode(), rho, u, phi, C, nullptr, c->stream));
    c->launches++;
    return 0;
}

int lbm_get_force(lbm_ctx* c, void* F) {
    if (!c) return fail(LBM_EINVAL, "ctx is NULL");
    if (!c->inited) return fail(LBM_ESTATE, "lbm_get_force before init");
    if (!F) return fail(LBM_EINVAL, "F is NULL");
    DeviceGuard g(c->device);
    if (c->sh.sc && c->psi_t != c->t) { int rc = run_psi(c); if (rc) return rc; }
    CK(c->ops->macros(c->kp(), c->model, (int)(c->t & 1), c->wmode(), nullptr, nullptr, nullptr, nullptr, F, c->stream));
    c->launches++;
    return 0;
}

size_t lbm_population_count(const lbm_ctx* c) {
    if (!c) return 0;
    return (size_t)c->sh.S * c->sh.Q * c->sh.N + (c->sh.scalar ? (size_t)c->sh.Qs * c->sh.N : 0);
}

int lbm_get_populations(lbm_ctx* c, void* f) {
    if (!c || !f) return fail(LBM_EINVAL, "NULL argument");
    if (!c->inited) return fail(LBM_ESTATE, "lbm_get_populations before init");
    DeviceGuard g(c->device);
    { int rs = tile_status_seen(c); if (rs) return rs; }
    const size_t nf = (size_t)c->sh.S * c->sh.Q * c->sh.N * c->sh.B, nh = (size_t)c->sh.Qs * c->sh.N * c->sh.B;
    if ((c->t & 1) == 0) {
        CK(cudaMemcpyAsync(f, c->f, nf, cudaMemcpyDeviceToDevice, c->stream));
        if (c->sh.scalar) CK(cudaMemcpyAsync((char*)f + nf, c->h, nh, cudaMemcpyDeviceToDevice, c->stream));
    } else {
        CK(c->ops->permute(c->kp(), c->model, 1, c->wmode(), f, 1, c->stream));
        c->launches += c->sh.scalar ? 2 : 1;
    }
    return 0;
}

int lbm_set_populations(lbm_ctx* c, const void* f) {
    if (!c || !f) return fail(LBM_EINVAL, "NULL argument");
    DeviceGuard g(c->device);
    const size_t nf = (size_t)c->sh.S * c->sh.Q * c->sh.N * c->sh.B, nh = (size_t)c->sh.Qs * c->sh.N * c->sh.B;
    CK(cudaMemcpyAsync(c->f, f, nf, cudaMemcpyDeviceToDevice, c->stream));
    if (c->sh.scalar) CK(cudaMemcpyAsync(c->h, (const char*)f + nf, nh, cudaMemcpyDeviceToDevice, c->stream));
    c->inited = true;
    c->t = 0;
    c->psi_t = -1;
    return 0;
}

int lbm_run_host(lbm_ctx* c, const void* f_in_host, int n, void* rho_h, void* u_h, void* phi_h, void* C_h) {
    if (!c) return fail(LBM_EINVAL, "ctx is NULL");
    if (C_h && !c->sh.scalar) return fail(LBM_EINVAL, "model has no scalar lattice");
    if (n < 0) return fail(LBM_EINVAL, "n < 0");
    DeviceGuard g(c->device);
    const Shape& sh = c->sh;
    if (f_in_host) {
        const size_t nf = (size_t)sh.S * sh.Q * sh.N * sh.B, nh = (size_t)sh.Qs * sh.N * sh.B;
        CK(cudaMemcpyAsync(c->f, f_in_host, nf, cudaMemcpyHostToDevice, c->stream));
        if (sh.scalar) CK(cudaMemcpyAsync(c->h, (const char*)f_in_host + nf, nh, cudaMemcpyHostToDevice, c->stream));
        c->inited = true;
        c->t = 0;
        c->psi_t = -1;
    }
    if (!c->inited) return fail(LBM_ESTATE, "lbm_run_host without populations");
    int rc = lbm_step(c, n);
    if (rc) return rc;
    if (rho_h || u_h || phi_h || C_h) {
        const size_t fb = sh.N * sh.B;
        const size_t need = (size_t)(sh.S + sh.d + 2) * fb;
        rc = ensure_scratch(c, need);
        if (rc) return rc;
        char* s = (char*)c->scratch;
        void* rho_d = rho_h ? s : nullptr;
        void* u_d = u_h ? s + (size_t)sh.S * fb : nullptr;
        void* phi_d = phi_h ? s + (size_t)(sh.S + sh.d) * fb : nullptr;
        void* C_d = C_h ? s + (size_t)(sh.S + sh.d + 1) * fb : nullptr;
        rc = lbm_get_macros(c, rho_d, u_d, phi_d, C_d);
        if (rc) return rc;
        if (rho_h) CK(cudaMemcpyAsync(rho_h, rho_d, (size_t)sh.S * fb, cudaMemcpyDeviceToHost, c->stream));
        if (u_h) CK(cudaMemcpyAsync(u_h, u_d, (size_t)sh.d * fb, cudaMemcpyDeviceToHost, c->stream));
        if (phi_h) CK(cudaMemcpyAsync(phi_h, phi_d, fb, cudaMemcpyDeviceToHost, c->stream));
        if (C_h) CK(cudaMemcpyAsync(C_h, C_d, fb, cudaMemcpyDeviceToHost, c->stream));
    }
    CK(cudaStreamSynchronize(c->stream));
    return tile_status(c);
}

int lbm_kernel_timing(lbm_ctx* c, int enable) {
    if (!c) return fail(LBM_EINVAL, "ctx is NULL");
    DeviceGuard g(c->device);
    CK(cudaStreamSynchronize(c->stream));
    drop_events(c);
    c->timing = enable != 0;
    return 0;
}

int lbm_kernel_time_ms(lbm_ctx* c, int kind, double* total_ms, int64_t* launches) {
    if (!c || !total_ms || !launches) return fail(LBM_EINVAL, "NULL argument");
    if (kind != 0 && kind != 1) return fail(LBM_EINVAL, "kind must be 0 (fused step) or 1 (psi pass)");
    DeviceGuard g(c->device);
    CK(cudaStreamSynchronize(c->stream));
    double sum = 0.0;
    const std::vector<cudaEvent_t>& v = c->ev[kind];
    for (size_t k = 0; k + 1 < v.size(); k += 2) {
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, v[k], v[k + 1]));
        sum += (double)ms;
    }
    *total_ms = sum;
    *launches = (int64_t)(v.size() / 2);
    return 0;
}

int lbm_set_path(lbm_ctx* c, int path, int rows_per_pencil) {
    if (!c) return fail(LBM_EINVAL, "ctx is NULL");
    DeviceGuard g(c->device);
    if (path == LBM_PATH_REGISTER) {
        CK(cudaStreamSynchronize(c->stream));
        tile_free(c);
        c->path_user_set = true;
        return 0;
    }
    if (path != LBM_PATH_PIPELINE) return fail(LBM_EINVAL, "unknown path");
    if (const char* why = tile_ineligible(c)) return fail(LBM_EINVAL, why);
    int rc = path_setup(c, rows_per_pencil);
    if (rc == 0) c->path_user_set = true;
    return rc;
}

int lbm_get_path(const lbm_ctx* c) { return c ? c->path : LBM_EINVAL; }

int lbm_set_mask(lbm_ctx* c, const unsigned char* mask) {
    if (!c) return fail(LBM_EINVAL, "ctx is NULL");
    // at an odd time level the in-place layout depends on which neighbours reflect: the mask may only change
    // when the populations sit in their own cells
    if (c->inited && (c->t & 1)) return fail(LBM_ESTATE, "lbm_set_mask needs an even time level (lbm_time)");
    DeviceGuard g(c->device);
    CK(cudaStreamSynchronize(c->stream));
    if (mask && c->path != LBM_PATH_REGISTER) tile_free(c);     // a solid-node mask runs on LBM_PATH_REGISTER only
    c->kp64.mask = mask;
    c->kp32.mask = mask;
    c->psi_t = -1;
    c->walls = c->bc_walls || mask != nullptr;
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }   // the graph holds the old parameters
    return 0;
}

int lbm_tile_schedule(int nm, int ns, int rows_per_pencil, int wrap_m, int wrap_s, int delay_rows, int32_t* items,
                      size_t capacity, size_t* count, int* deferred_rows) {
    if (!count) return fail(LBM_EINVAL, "count is NULL");
    if (nm < 1 || ns < 1) return fail(LBM_EINVAL, "nm and ns must be >= 1");
    int deferred = 0;
    const std::vector<lbm::TileRow> v = lbm::tile_schedule(nm, ns, rows_per_pencil, wrap_m != 0, wrap_s != 0, delay_rows, &deferred);
    *count = v.size();
    if (deferred_rows) *deferred_rows = deferred;
    if (items) {
        if (capacity < v.size()) return fail(LBM_EINVAL, "capacity too small");
        for (size_t k = 0; k < v.size(); ++k) {
            items[3 * k + 0] = v[k].kind;
            items[3 * k + 1] = v[k].m;
            items[3 * k + 2] = v[k].s;
        }
    }
    return 0;
}

int lbm_tile_tickets(int nm, int ns, int nxs, int rows_per_pencil, int wrap_m, int wrap_s, int delay_rows, int three_d,
                     int32_t* tickets, size_t capacity, size_t* count) {
    if (!count) return fail(LBM_EINVAL, "count is NULL");
    if (nm < 1 || ns < 1 || nxs < 1) return fail(LBM_EINVAL, "nm, ns and nxs must be >= 1");
    const std::vector<lbm::TileRow> rows = lbm::tile_schedule(nm, ns, rows_per_pencil, wrap_m != 0, wrap_s != 0, delay_rows, nullptr);
    const std::vector<lbm::TileItem> v = lbm::tile_tickets(rows, nxs, three_d != 0);
    *count = v.size();
    if (tickets) {
        if (capacity < v.size()) return fail(LBM_EINVAL, "capacity too small");
        static_assert(sizeof(lbm::TileItem) == 8 * sizeof(int32_t), "ticket layout");
        std::memcpy(tickets, v.data(), v.size() * sizeof(lbm::TileItem));
    }
    return 0;
}

int lbm_check(lbm_ctx* c) {
    if (!c) return fail(LBM_EINVAL, "ctx is NULL");
    DeviceGuard g(c->device);
    CK(cudaStreamSynchronize(c->stream));
    return tile_status(c);
}

#ifdef LBM_TILE_TRACE
int lbm_debug_trace(void* out) { return (int)cudaMemcpy(out, g_trace, sizeof(long long) * 10 * 4096, cudaMemcpyDeviceToHost); }
#endif

// ---------------------------------------------------------------------------------------------------------------
// lbm_step_static: the Shan-Chen step for callers that must not allocate (include/lbm.h).  The psi field -- the scratch
// of the psi pass / fused step pair -- lives in a file-scope device array instead of a workspace.  In HOST code the
// array's name is only a stand-in for the symbol: its device address comes from cudaGetSymbolAddress, once per device.
// ---------------------------------------------------------------------------------------------------------------
}  // extern "C"

#define LBM_STATIC_SCRATCH_BYTES (16u << 20)
static __device__ __align__(256) unsigned char g_static_scratch[LBM_STATIC_SCRATCH_BYTES];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
void* g_static_ptr[STATIC_MAX_DEVICES];           // device address of g_static_scratch per device ordinal (nullptr: not asked yet)
std::mutex g_static_mutex;

// the device address of the scratch array on the CURRENT device
int static_scratch_address(void** out) {
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return fail(LBM_EINVAL, "lbm_step_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        void* ptr = nullptr;
        CK(cudaGetSymbolAddress(&ptr, g_static_scratch));
        g_static_ptr[dev] = ptr;
    }
    *out = g_static_ptr[dev];
    return 0;
}
}  // namespace

extern "C" {

size_t lbm_static_scratch_bytes(void) { return (size_t)LBM_STATIC_SCRATCH_BYTES; }

int lbm_step_static(int nx, int ny, int nz, int lattice, int model, const lbm_params* p, void* f, int n) {
    Shape sh;
    const std::string e = validate(nx, ny, nz, lattice, model, p, &sh);
    if (!e.empty()) return fail(LBM_EINVAL, "lbm_step_static: " + e);
    if (!f) return fail(LBM_EINVAL, "lbm_step_static: f is NULL");
    if (!sh.sc) return fail(LBM_EINVAL, "lbm_step_static: the model has no psi field (no scratch): use lbm_step");
    if (n < 0 || (n & 1)) return fail(LBM_EINVAL, "lbm_step_static: n must be even and >= 0 (the populations are canonical at even time levels)");
    const size_t need = (size_t)sh.S * sh.N * sh.B;
    if (need > (size_t)LBM_STATIC_SCRATCH_BYTES)
        return fail(LBM_EINVAL, "lbm_step_static: the psi field needs " + std::to_string(need) + " bytes, the static scratch holds " +
                                    std::to_string((size_t)LBM_STATIC_SCRATCH_BYTES) + " (S * nx * ny * nz * sizeof(value)): use lbm_create / lbm_step");
    void* scratch = nullptr;
    int rc = static_scratch_address(&scratch);
    if (rc) return rc;
    // a context on the stack: no workspace, no schedule, no graph -- only what fill_kp and the launchers read
    lbm_ctx c{};
    c.nx = nx; c.ny = ny; c.nz = nz; c.lattice = lattice; c.model = model;
    c.p = *p; c.sh = sh;
    c.stream = (cudaStream_t)p->stream;
    c.f = f;
    c.h = sh.scalar ? (char*)f + (size_t)sh.S * sh.Q * sh.N * sh.B : nullptr;     // canonical layout: h follows f
    c.psi = scratch;
    c.bc_walls = p->bc[0] || p->bc[1] || p->bc[2];
    c.forced = p->forcing == 1 ? 2 : 1;
    if (p->precision == 64) c.ops = lattice == LBM_D3Q19 ? lbm::ops_f64_d3q19() : lbm::ops_f64_d2q9();
    else c.ops = lattice == LBM_D3Q19 ? lbm::ops_f32_d3q19() : lbm::ops_f32_d2q9();
    fill_kp(c.kp64, &c);
    fill_kp(c.kp32, &c);
    const int wmode = c.bc_walls ? 1 : 0;
    int moving = 0;
    for (int a = 0; a < 3; ++a)
        for (int sd = 0; sd < 2; ++sd)
            for (int b = 0; b < 3; ++b)
                if (p->bc[a] == 1 && p->wall_u[a][sd][b] != 0.0) moving = 1;
    for (int k = 0; k < n; ++k) {
        // a2 writes psi of every cell before a3 reads any: nothing in the scratch needs to start at zero
        CK(c.ops->psi(c.kp(), model, k & 1, wmode, c.stream));
        CK(c.ops->step(c.kp(), model, k & 1, wmode, c.forced, moving, c.stream));
    }
    return 0;
}

int64_t lbm_time(const lbm_ctx* c) { return c ? c->t : -1; }
int64_t lbm_launch_count(const lbm_ctx* c) { return c ? c->launches : -1; }

int lbm_lattice_table(int lattice, int kind, int* Q, int* cc, double* w, int* opp) {
    if (!Q || !cc || !w || !opp) return fail(LBM_EINVAL, "NULL argument");
    if (lattice != LBM_D2Q9 && lattice != LBM_D3Q19) return fail(LBM_EINVAL, "unknown lattice");
    auto fill = [&](auto L, bool flow, double w0) {
        using LL = decltype(L);
        *Q = LL::Q;
        for (int i = 0; i < LL::Q; ++i) {
            for (int a = 0; a < 3; ++a) cc[3 * i + a] = LL::c(i, a);
            opp[i] = LL::opp(i);
            if (!flow) w[i] = i == 0 ? w0 : (1.0 - w0) / (double)(LL::Q - 1);
        }
    };
    if (kind == 0) {
        if (lattice == LBM_D3Q19) { fill(lbm::D3Q19{}, true, 0); for (int i = 0; i < 19; ++i) w[i] = lbm::D3Q19::w(i); }
        else { fill(lbm::D2Q9{}, true, 0); for (int i = 0; i < 9; ++i) w[i] = lbm::D2Q9::w(i); }
    } else {
        if (lattice == LBM_D3Q19) fill(lbm::D3Q7{}, false, 0.25); else fill(lbm::D2Q5{}, false, 0.4);
    }
    return 0;
}

}  // extern "C"
