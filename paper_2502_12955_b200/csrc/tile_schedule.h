// Host-side row schedule of the resident-tile kernel (tile.cuh): the order in which one launch works through the
// rows of one time step of a Shan-Chen model.
//
// Why: psi^sigma(x + c_i, t) must be known for all neighbours before cell x is collided (Eq. 11 / 13,
// PAPER.md:128, 136; R9), and psi(t + 1) of a cell can only be formed once the step of all its neighbours
// has written the populations that stream into it (Eq. 5 / 7).  One launch therefore does two things per row:
//
//   STEP item  the fused step a1, a3-a8 of time level t for the row, reading psi(t) (complete: it was written by the
//              previous launch).  STEP items depend on nothing inside the launch; they come in pencil order: pencils of
//              `py` rows of the slower-but-one axis, marched along the slowest axis.
//   PSI item   step a2 for time level t + 1: rho^sigma(t + 1) of the row from the populations the STEP items of the 3 x 3
//              rows around it (periodic wrap; none beyond a wall) have just written, psi(t + 1) to the OTHER psi
//              buffer.  It becomes ready when the last of those STEP items is done and is
//              listed `delay` STEP rows later: by then the blocks that took those STEP items (the list is dealt out
//              round-robin) have long finished them, so the block that takes the PSI item does not wait, and the
//              populations are still in L2 (the distance is one plane of the pencil, py + 1 rows, plus the delay).
//              The rows at the edge of a pencil wait for the neighbouring pencil and are read from HBM again (a
//              fraction 1 / py of the rows in 3D, none in 2D).
//
// Row coordinates: (m, s) = (y, z) for D3Q19; (0, y) for D2Q9 (the marching axis is always the slowest one).
#pragma once
#include <cstdint>
#include <vector>

namespace lbm {

enum { TILE_STEP = 0, TILE_PSI = 1 };

struct TileRow {
    int32_t kind, m, s;
};

// py: rows per pencil (clamped to [1, nm]); wrap_m / wrap_s: that axis is periodic (else: walls, no neighbour beyond).
// Returns the merged list (2 * nm * ns items): the STEP rows in pencil order; a PSI row that the k-th STEP row completes
// comes right after STEP row k + delay (all that are left after the last STEP row).
// *deferred_rows (optional): PSI rows that become ready more than 2 * py + 8 STEP rows after their own STEP row (they
// wait for another pencil or for the wrapped plane: their populations have left L2 by then).
inline std::vector<TileRow> tile_schedule(int nm, int ns, int py, bool wrap_m, bool wrap_s, int delay, int* deferred_rows) {
    std::vector<TileRow> items;
    if (deferred_rows) *deferred_rows = 0;
    if (nm < 1 || ns < 1) return items;
    if (py < 1) py = 1;
    if (py > nm) py = nm;
    const size_t R = (size_t)nm * ns;
    auto nbr = [](int v, int d, int n, bool wrap, int* out) {
        int q = v + d;
        if (q < 0 || q >= n) {
            if (!wrap) return false;
            q = q < 0 ? q + n : q - n;
            if (q < 0 || q >= n) return false;      // n == 1: the only row is its own neighbour
        }
        *out = q;
        return true;
    };
    // the (up to 9, possibly coinciding) rows around (m, s), itself included
    auto around = [&](int m, int s, int (*out)[2]) {
        int n = 0;
        for (int ds = -1; ds <= 1; ++ds)
            for (int dm = -1; dm <= 1; ++dm) {
                int mm, ss;
                if (!nbr(m, dm, nm, wrap_m, &mm) || !nbr(s, ds, ns, wrap_s, &ss)) continue;
                bool dup = false;
                for (int k = 0; k < n; ++k) dup = dup || (out[k][0] == mm && out[k][1] == ss);
                if (!dup) { out[n][0] = mm; out[n][1] = ss; ++n; }
            }
        return n;
    };
    if (delay < 0) delay = 0;
    struct Ready { int32_t m, s; int64_t at; };
    std::vector<Ready> fifo;                 // PSI rows that are ready, in the order they became ready
    size_t head = 0;
    std::vector<uint8_t> stepped(R, 0), listed(R, 0);
    std::vector<int64_t> step_pos(R, 0);
    items.reserve(2 * R);
    int64_t n_step = 0;
    for (int m0 = 0; m0 < nm; m0 += py) {
        const int rows = (m0 + py <= nm ? py : nm - m0);
        for (int s = 0; s < ns; ++s)
            for (int m = m0; m < m0 + rows; ++m) {
                items.push_back(TileRow{TILE_STEP, m, s});
                stepped[(size_t)s * nm + m] = 1;
                step_pos[(size_t)s * nm + m] = n_step++;
                int q[9][2], r[9][2];
                const int nq = around(m, s, q);
                for (int k = 0; k < nq; ++k) {
                    const size_t qi = (size_t)q[k][1] * nm + q[k][0];
                    if (listed[qi]) continue;
                    const int nr = around(q[k][0], q[k][1], r);
                    bool ready = true;
                    for (int j = 0; j < nr; ++j) ready = ready && stepped[(size_t)r[j][1] * nm + r[j][0]];
                    if (!ready) continue;
                    listed[qi] = 1;
                    fifo.push_back(Ready{q[k][0], q[k][1], n_step - 1});
                    if (deferred_rows && n_step - 1 - step_pos[qi] > 2 * (int64_t)py + 8) ++*deferred_rows;
                }
                for (; head < fifo.size() && fifo[head].at + delay <= n_step - 1; ++head)
                    items.push_back(TileRow{TILE_PSI, fifo[head].m, fifo[head].s});
            }
    }
    for (; head < fifo.size(); ++head) items.push_back(TileRow{TILE_PSI, fifo[head].m, fifo[head].s});
    return items;
}

// One ticket of the resident-tile kernel: a tile to step and / or a tile whose psi(t + 1) is due
struct TileItem {
    int sx, sy, sz, sv;               // STEP part: x-segment, row of the tile to step; sv != 0: present
    int px, py, pz, pv;               // PSI part: the tile whose psi(t + 1) is formed; pv != 0: present
};

// The tickets of one time step from the row schedule: ticket k carries the k-th tile to step (rows in schedule order,
// nxs tiles per row, x fastest) and the next tile whose psi is due.  A PSI row is due where the schedule lists it --
// every step it depends on is the STEP part of an EARLIER ticket, which is what makes the kernel's waits deadlock-free
// -- so a PSI tile rides on the first ticket whose index is at least the number of tiles stepped before its row was
// listed; the PSI tiles left over after the last step form a tail of PSI-only tickets.  three_d: rows are (y, z) = (m, s),
// else (y, z) = (s, 0).
inline std::vector<TileItem> tile_tickets(const std::vector<TileRow>& rows, int nxs, bool three_d) {
    struct Pos { int xs, y, z; size_t due; };
    std::vector<Pos> steps, psis;
    for (const TileRow& r : rows) {
        Pos q;
        q.y = three_d ? r.m : r.s;
        q.z = three_d ? r.s : 0;
        q.due = steps.size();                 // PSI: may ride on the step ticket with this index or a later one
        for (int xs = 0; xs < nxs; ++xs) { q.xs = xs; (r.kind == TILE_STEP ? steps : psis).push_back(q); }
    }
    std::vector<TileItem> items;
    items.reserve(steps.size() + steps.size() / 8 + 16);
    size_t jp = 0;
    for (size_t k = 0; k < steps.size() || jp < psis.size(); ++k) {
        TileItem it = {0, 0, 0, 0, 0, 0, 0, 0};
        if (k < steps.size()) { it.sx = steps[k].xs; it.sy = steps[k].y; it.sz = steps[k].z; it.sv = 1; }
        if (jp < psis.size() && (psis[jp].due <= k || k >= steps.size())) {
            it.px = psis[jp].xs; it.py = psis[jp].y; it.pz = psis[jp].z; it.pv = 1;
            ++jp;
        }
        items.push_back(it);
    }
    return items;
}

}  // namespace lbm
