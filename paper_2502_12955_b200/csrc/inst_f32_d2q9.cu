// kernel instances: precision float, flow lattice D2Q9
#include "inst.cuh"
namespace lbm {
const Ops* ops_f32_d2q9() { return Launch<float, D2Q9>::ops(); }
}  // namespace lbm
