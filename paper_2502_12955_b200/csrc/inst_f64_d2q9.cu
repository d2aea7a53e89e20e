// kernel instances: precision double, flow lattice D2Q9
#include "inst.cuh"
namespace lbm {
const Ops* ops_f64_d2q9() { return Launch<double, D2Q9>::ops(); }
}  // namespace lbm
