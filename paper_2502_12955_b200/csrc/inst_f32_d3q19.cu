// kernel instances: precision float, flow lattice D3Q19
#include "inst.cuh"
namespace lbm {
const Ops* ops_f32_d3q19() { return Launch<float, D3Q19>::ops(); }
}  // namespace lbm
