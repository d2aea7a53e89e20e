// Host-side row schedule of the resident-tile kernel (tile.cuh): the order in which one launch works through the
// rows of one time step of a Shan-Chen model.
//
// Why: psi^sigma(x + c_i, t) must be known for all neighbours before cell x is collided (Eq. 11 / 13,
// PAPER.md:128, 136; R9), and with in-place streaming a cell's populations can only be read before its
// own step overwrites them.  The resident-tile kernel loads the populations of a tile ONCE into shared memory,
// computes and publishes its psi (step a2), keeps the tile resident until the psi of the tiles around it has been
// published by the blocks that own them, and then collides and streams it (a1, a3-a8) from shared memory.
//
// A FULL row item is one such load-psi-wait-step life cycle for every tile of the row.  The step of row (m, s)
// needs psi of the 3 x 3 rows around it.  Rows whose own FULL item comes within `window` rows after it provide
// their psi in time by themselves; any other needed row that has not been computed yet in this launch (the wrapped
// neighbour plane at the start of a pencil, the first row of the next pencil) gets a PSI_ONLY item first: its flow
// populations are loaded, psi is computed and published, and the tile is dropped -- its FULL item comes later and
// reads the populations a second time (a fraction 1 / rows_per_pencil of the rows in 3D, one row in 2D).
//
// Row coordinates: (m, s) = (y, z) for D3Q19; (0, y) for D2Q9 (the marching axis is always the slowest one).
#pragma once
#include <cstdint>
#include <vector>

namespace lbm {

enum { TILE_FULL = 0, TILE_PSI_ONLY = 1 };

struct TileRow {
    int32_t kind, m, s;
};

// py: rows per pencil (clamped to [1, nm]); wrap_m / wrap_s: that axis is periodic (else: walls, no neighbour beyond).
// *lead_rows (optional): the largest distance, in items of the returned list, from a FULL item to the LAST item that
// provides a psi row it needs and comes after it -- what the kernel's pipeline depth must cover (tile.cuh).
inline std::vector<TileRow> tile_schedule(int nm, int ns, int py, bool wrap_m, bool wrap_s, int* lead_rows) {
    std::vector<TileRow> items;
    if (lead_rows) *lead_rows = 0;
    if (nm < 1 || ns < 1) return items;
    if (py < 1) py = 1;
    if (py > nm) py = nm;
    struct MS { int m, s; };
    std::vector<MS> order;
    order.reserve((size_t)nm * ns);
    std::vector<int64_t> pos_full((size_t)nm * ns, 0);
    std::vector<int> window((size_t)nm * ns, 0);
    for (int m0 = 0; m0 < nm; m0 += py) {
        const int rows = (m0 + py <= nm ? py : nm - m0);
        for (int s = 0; s < ns; ++s)
            for (int m = m0; m < m0 + rows; ++m) {
                pos_full[(size_t)s * nm + m] = (int64_t)order.size();
                window[(size_t)s * nm + m] = rows + 1;      // FULL(m + 1, s + 1) comes rows + 1 items after FULL(m, s)
                order.push_back(MS{m, s});
            }
    }
    auto nbr = [](int v, int d, int n, bool wrap, int* out) {
        int q = v + d;
        if (q < 0 || q >= n) {
            if (!wrap) return false;
            q = q < 0 ? q + n : q - n;
        }
        *out = q;
        return true;
    };
    std::vector<uint8_t> have((size_t)nm * ns, 0);
    std::vector<int64_t> provider((size_t)nm * ns, -1);    // position of the first item that computes psi of the row
    items.reserve(order.size() + order.size() / (size_t)py + 64);
    for (size_t idx = 0; idx < order.size(); ++idx) {
        const MS r = order[idx];
        for (int ds = -1; ds <= 1; ++ds)
            for (int dm = -1; dm <= 1; ++dm) {
                int mm, ss;
                if (!nbr(r.m, dm, nm, wrap_m, &mm) || !nbr(r.s, ds, ns, wrap_s, &ss)) continue;
                const size_t k = (size_t)ss * nm + mm;
                if (have[k]) continue;
                const int64_t d = pos_full[k] - (int64_t)idx;
                if (d >= 0 && d <= window[(size_t)r.s * nm + r.m]) continue;     // its own FULL item comes soon enough
                have[k] = 1;
                provider[k] = (int64_t)items.size();
                items.push_back(TileRow{TILE_PSI_ONLY, mm, ss});
            }
        const size_t k = (size_t)r.s * nm + r.m;
        if (!have[k]) { have[k] = 1; provider[k] = (int64_t)items.size(); }
        items.push_back(TileRow{TILE_FULL, r.m, r.s});
    }
    if (lead_rows) {
        int64_t lead = 0;
        for (size_t p = 0; p < items.size(); ++p) {
            if (items[p].kind != TILE_FULL) continue;
            for (int ds = -1; ds <= 1; ++ds)
                for (int dm = -1; dm <= 1; ++dm) {
                    int mm, ss;
                    if (!nbr(items[p].m, dm, nm, wrap_m, &mm) || !nbr(items[p].s, ds, ns, wrap_s, &ss)) continue;
                    const int64_t d = provider[(size_t)ss * nm + mm] - (int64_t)p;
                    if (d > lead) lead = d;
                }
        }
        *lead_rows = (int)lead;
    }
    return items;
}

}  // namespace lbm
