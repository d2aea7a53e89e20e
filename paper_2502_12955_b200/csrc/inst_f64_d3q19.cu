// kernel instances: precision double, flow lattice D3Q19
#include "inst.cuh"
namespace lbm {
const Ops* ops_f64_d3q19() { return Launch<double, D3Q19>::ops(); }
}  // namespace lbm
