// Host-side row schedule of the pipelined kernel (pipe.cuh): the order in which one launch works through the
// psi rows (step a2) and the step rows (a1, a3-a8) of one time step of a Shan-Chen model.
//
// Why: psi^sigma(x + c_i, t) must be known for all neighbours before cell x is collided (Eq. 11 / 13,
// PAPER.md:128, 136; R9), and with in-place streaming a cell's populations can only be read
// before its own step overwrites them.  A separate psi pass re-reads every population from HBM.  Here both
// passes run in ONE launch as a list of row items: a psi item reads the populations of a row (first touch,
// from HBM) and publishes psi; the step item of the same row follows a short distance later and finds the
// populations in L2.  The only rule the order must obey: every psi row a step row needs (its own row and the
// rows around it, periodic wrap) comes EARLIER in the list, and a row's psi item comes before its step item.
// Any traversal of the step rows satisfies it by construction below; the traversal chosen (pencils of `py`
// rows, marched along the slow axis) only sets the reuse distance in L2.
//
// Row coordinates: (m, s) = (y, z) for D3Q19; (0, y) for D2Q9 (the marching axis is always the slowest one).
#pragma once
#include <cstdint>
#include <vector>

namespace lbm {

struct WaveItem {
    int32_t m;      // bit 31 set: psi row, clear: step row
    int32_t s;
};
constexpr int32_t WAVE_PSI_BIT = (int32_t)0x80000000u;

// py: rows per pencil (>= 1); lead: how many step rows ahead the psi rows are issued (>= 0)
inline std::vector<WaveItem> wave_schedule(int nm, int ns, int py, int lead) {
    std::vector<WaveItem> items;
    if (nm < 1 || ns < 1) return items;
    if (py < 1) py = 1;
    if (py > nm) py = nm;
    if (lead < 0) lead = 0;
    std::vector<WaveItem> order;
    order.reserve((size_t)nm * ns);
    for (int m0 = 0; m0 < nm; m0 += py)
        for (int s = 0; s < ns; ++s)
            for (int m = m0; m < m0 + py && m < nm; ++m) order.push_back(WaveItem{m, s});
    std::vector<uint8_t> done((size_t)nm * ns, 0);
    items.reserve(2 * order.size());
    auto wrap = [](int v, int n) { return v < 0 ? v + n : (v >= n ? v - n : v); };
    const size_t n = order.size();
    for (size_t j = 0; j < n + (size_t)lead; ++j) {
        if (j < n) {
            const WaveItem r = order[j];
            for (int ds = -1; ds <= 1; ++ds)
                for (int dm = -1; dm <= 1; ++dm) {
                    const int mm = wrap(r.m + dm, nm), ss = wrap(r.s + ds, ns);
                    uint8_t& d = done[(size_t)ss * nm + mm];
                    if (!d) {
                        d = 1;
                        items.push_back(WaveItem{mm | WAVE_PSI_BIT, ss});
                    }
                }
        }
        if (j >= (size_t)lead) items.push_back(order[j - (size_t)lead]);
    }
    return items;
}

}  // namespace lbm
