// See gather_tables.h.  Pure host C++.
#include "gather_tables.h"

#include <algorithm>

namespace hub {

namespace {

struct Edge {
    int row;        // 0..G-1 within the group
    int bank;       // col % G
    uint32_t entry; // col * 2 + neg
    int color;
};

// Proper edge colouring of a bipartite multigraph (rows x banks) with C colours,
// C >= max degree (Koenig): alternating-path recolouring.
void edge_colour(std::vector<Edge> &edges, int G, int C)
{
    std::vector<int> rowc((size_t)G * C, -1), bankc((size_t)G * C, -1);   // [vertex][colour] -> edge id
    for (int e = 0; e < (int)edges.size(); ++e) {
        const int u = edges[e].row, v = edges[e].bank;
        int a = 0, b = 0;
        while (rowc[(size_t)u * C + a] >= 0) ++a;
        while (bankc[(size_t)v * C + b] >= 0) ++b;
        if (a != b && bankc[(size_t)v * C + a] >= 0) {
            // free colour a at bank v: swap a <-> b along the alternating path that starts at v with colour a
            std::vector<int> path;
            bool at_bank = true;
            int vert = v, col = a;
            for (;;) {
                int f = at_bank ? bankc[(size_t)vert * C + col] : rowc[(size_t)vert * C + col];
                if (f < 0) break;
                path.push_back(f);
                vert = at_bank ? edges[f].row : edges[f].bank;
                at_bank = !at_bank;
                col = (col == a) ? b : a;
            }
            for (int f : path) {
                rowc[(size_t)edges[f].row * C + edges[f].color] = -1;
                bankc[(size_t)edges[f].bank * C + edges[f].color] = -1;
            }
            for (int f : path) {
                edges[f].color = (edges[f].color == a) ? b : a;
                rowc[(size_t)edges[f].row * C + edges[f].color] = f;
                bankc[(size_t)edges[f].bank * C + edges[f].color] = f;
            }
        }
        edges[e].color = a;
        rowc[(size_t)u * C + a] = e;
        bankc[(size_t)v * C + a] = e;
    }
}

}  // namespace

void build_gather_table(const SpinTable &tab, int lanes, int64_t zero_base, GatherTable &out)
{
    const int64_t dim = tab.dim;
    out.ld = (dim + 31) / 32 * 32;
    out.w = (std::max(tab.width, 1) + kSlotBatch - 1) / kSlotBatch * kSlotBatch;
    out.cnt.assign((size_t)dim, 0);
    out.conflicts = 0;
    const uint32_t pad0 = (uint32_t)zero_base * 2u;
    out.ent.assign((size_t)out.ld * out.w, pad0);
    auto put = [&](int64_t i, int k, uint32_t e) { out.ent[((size_t)(k / kSlotBatch) * out.ld + i) * kSlotBatch + k % kSlotBatch] = e; };
    auto entry_of = [&](size_t s) { return (uint32_t)tab.col[s] * 2u + (tab.plus[s] ? 0u : 1u); };

    if (lanes <= 0) {
        for (int64_t r = 0; r < dim; ++r) {
            const int n = (int)(tab.rowptr[r + 1] - tab.rowptr[r]);
            out.cnt[(size_t)r] = n;
            for (int k = 0; k < n; ++k) put(r, k, entry_of((size_t)(tab.rowptr[r] + k)));
        }
        return;
    }
    const int G = lanes;
    std::vector<Edge> edges;
    std::vector<int> bank_deg(G), used;
    for (int64_t w0 = 0; w0 < dim; w0 += 32) {
        const int64_t w1 = std::min(dim, w0 + 32);
        int nmax = 0;
        for (int64_t r = w0; r < w1; ++r) nmax = std::max(nmax, (int)(tab.rowptr[r + 1] - tab.rowptr[r]));
        const int W = std::max(kSlotBatch, (nmax + kSlotBatch - 1) / kSlotBatch * kSlotBatch);   // slots the warp walks
        for (int64_t g0 = w0; g0 < w1; g0 += G) {
            const int64_t g1 = std::min(w1, g0 + G);
            edges.clear();
            std::fill(bank_deg.begin(), bank_deg.end(), 0);
            for (int64_t r = g0; r < g1; ++r)
                for (int64_t s = tab.rowptr[r]; s < tab.rowptr[r + 1]; ++s) {
                    Edge e{(int)(r - g0), (int)(tab.col[(size_t)s] % G), entry_of((size_t)s), -1};
                    ++bank_deg[e.bank];
                    edges.push_back(e);
                }
            const int C = std::max(W, *std::max_element(bank_deg.begin(), bank_deg.end()));
            edge_colour(edges, G, C);
            // slot occupancy [slot][bank] and [row][slot]
            std::vector<int> slot_bank((size_t)W * G, 0);
            std::vector<char> row_slot((size_t)G * W, 0);
            for (const Edge &e : edges)
                if (e.color < W) { ++slot_bank[(size_t)e.color * G + e.bank]; row_slot[(size_t)e.row * W + e.color] = 1; }
            // colours beyond the warp's slots (a bank with more entries than slots): fold back, conflict accepted
            for (Edge &e : edges) {
                if (e.color < W) continue;
                int best = -1, best_load = 1 << 30;
                for (int s = 0; s < W; ++s) {
                    if (row_slot[(size_t)e.row * W + s]) continue;
                    const int load = slot_bank[(size_t)s * G + e.bank];
                    if (load < best_load) { best_load = load; best = s; }
                }
                e.color = best;                       // a row has at most W entries, so a free slot exists
                ++slot_bank[(size_t)best * G + e.bank];
                row_slot[(size_t)e.row * W + best] = 1;
            }
            for (int s = 0; s < W; ++s)
                for (int b = 0; b < G; ++b)
                    if (slot_bank[(size_t)s * G + b] > 1) out.conflicts += slot_bank[(size_t)s * G + b];
            // write entries; holes of a row below its last used slot point at a zero slot on a free bank
            for (const Edge &e : edges) {
                const int64_t r = g0 + e.row;
                put(r, e.color, e.entry);
                out.cnt[(size_t)r] = std::max(out.cnt[(size_t)r], e.color + 1);
            }
            for (int64_t r = g0; r < g1; ++r) {
                const int rr = (int)(r - g0);
                for (int s = 0; s < out.cnt[(size_t)r]; ++s) {
                    if (row_slot[(size_t)rr * W + s]) continue;
                    int zb = 0;
                    for (int z = 0; z < G; ++z) {
                        const int b = (int)((zero_base + z) % G);
                        if (slot_bank[(size_t)s * G + b] == 0) { zb = z; break; }
                    }
                    ++slot_bank[(size_t)s * G + (int)((zero_base + zb) % G)];
                    put(r, s, (uint32_t)(zero_base + zb) * 2u);
                }
            }
        }
    }
}

}  // namespace hub
