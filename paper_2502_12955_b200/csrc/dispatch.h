// Host-side dispatch table: one Ops per (precision, flow lattice), each filled by its own
// translation unit (inst_*.cu) so the kernel variants compile in parallel.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lbm {

struct InitArgs;
struct TileArgs;

struct Ops {
    // kp points at a KP<R> of the matching precision
    cudaError_t (*psi)(const void* kp, int model, int parity, int walls, cudaStream_t st);
    cudaError_t (*step)(const void* kp, int model, int parity, int wmode, int forced, int moving, cudaStream_t st);
    cudaError_t (*macros)(const void* kp, int model, int parity, int walls, void* rho, void* u, void* phi, void* C,
                          void* F, cudaStream_t st);
    // canonical <-> slot permutation of the flow lattices (S of them) and of the scalar lattice
    cudaError_t (*permute)(const void* kp, int model, int parity, int walls, void* canon, int to_canonical,
                           cudaStream_t st);
    cudaError_t (*init)(const void* kp, int model, const InitArgs* ia, cudaStream_t st);
    // resident-tile persistent kernel of the Shan-Chen models (tile.cuh); walls: bounce-back walls in y and / or z
    cudaError_t (*tile)(const void* kp, int model, int parity, int walls, int vshift, const TileArgs* wa, int blocks, cudaStream_t st);
    int (*tile_blocks)(int model, int parity, int walls, int vshift);     // co-resident blocks on the current device
    int (*tile_tx)();                                         // cells per tile
};

const Ops* ops_f64_d2q9();
const Ops* ops_f64_d3q19();
const Ops* ops_f32_d2q9();
const Ops* ops_f32_d3q19();

}  // namespace lbm
