// Host-side preparation.  See host_tables.h.
#include "host_tables.h"

#include <algorithm>
#include <new>

namespace hub {

uint64_t binom(int n, int k)
{
    if (k < 0 || k > n || n < 0) return 0;
    if (k > n - k) k = n - k;
    uint64_t r = 1;
    for (int i = 1; i <= k; ++i) r = r * (uint64_t)(n - k + i) / (uint64_t)i;  // exact at every step
    return r;
}

int64_t rank_of(uint32_t s)
{
    // position in the ascending list of equal-popcount patterns: patterns that
    // are smaller agree on the bits above some set bit p_k and have a 0 there,
    // with the remaining k set bits placed among the p_k lower positions.
    int64_t r = 0;
    int k = 0;
    while (s) {
        int p = __builtin_ctz(s);
        ++k;
        r += (int64_t)binom(p, k);
        s &= s - 1;
    }
    return r;
}

// next larger integer with the same number of set bits (Gosper)
static inline uint64_t next_same_popcount(uint64_t v)
{
    uint64_t c = v & (~v + 1);
    uint64_t r = v + c;
    return (((r ^ v) >> 2) / c) | r;
}

int build_spin_table(int n_sites, int n_el, const int32_t *bonds, int n_bonds, SpinTable &out)
{
    if (n_sites < 1 || n_sites > 32 || n_el < 0 || n_el > n_sites || n_bonds < 0) return -1;
    if (n_bonds > 0 && !bonds) return -1;
    for (int b = 0; b < n_bonds; ++b) {
        int i = bonds[2 * b], j = bonds[2 * b + 1];
        if (i < 0 || j < 0 || i >= n_sites || j >= n_sites || i == j) return -1;
    }
    uint64_t dim = binom(n_sites, n_el);
    if (dim >= 0x7fffffffull) return -6;
    try {
        out.n_sites = n_sites;
        out.n_el = n_el;
        out.dim = (int64_t)dim;
        out.states.resize(dim);
        // ascending enumeration
        uint64_t s = (n_el == 0) ? 0 : ((n_el == 64) ? ~0ull : ((1ull << n_el) - 1));
        for (uint64_t r = 0; r < dim; ++r) {
            out.states[r] = (uint32_t)s;
            if (n_el > 0 && r + 1 < dim) s = next_same_popcount(s);
        }
        // per bond: mask of the sites strictly between its ends (reading Q4)
        std::vector<uint32_t> between(n_bonds);
        for (int b = 0; b < n_bonds; ++b) {
            int lo = std::min(bonds[2 * b], bonds[2 * b + 1]), hi = std::max(bonds[2 * b], bonds[2 * b + 1]);
            uint32_t below_hi = (hi == 0) ? 0u : (uint32_t)((1ull << hi) - 1);
            uint32_t upto_lo = (uint32_t)((1ull << (lo + 1)) - 1);
            between[b] = below_hi & ~upto_lo;
        }
        out.rowptr.assign(dim + 1, 0);
        // pass 1: count, pass 2: fill.  A hop exists on bond (i,j) for state s
        // when exactly one of the two sites is occupied; the state it connects
        // to is s with both bits flipped; H is symmetric so the same entry
        // serves as <s'|H|s> and <s|H|s'>; we store, for row s, column s'.
        int width = 0;
        for (uint64_t r = 0; r < dim; ++r) {
            uint32_t st = out.states[r];
            int cnt = 0;
            for (int b = 0; b < n_bonds; ++b) {
                uint32_t pair = (1u << bonds[2 * b]) | (1u << bonds[2 * b + 1]);
                uint32_t occ = st & pair;
                if (occ != 0 && occ != pair) ++cnt;
            }
            out.rowptr[r + 1] = out.rowptr[r] + cnt;
            width = std::max(width, cnt);
        }
        out.width = width;
        out.col.resize((size_t)out.rowptr[dim]);
        out.plus.resize((size_t)out.rowptr[dim]);
        for (uint64_t r = 0; r < dim; ++r) {
            uint32_t st = out.states[r];
            int64_t k = out.rowptr[r];
            for (int b = 0; b < n_bonds; ++b) {
                uint32_t pair = (1u << bonds[2 * b]) | (1u << bonds[2 * b + 1]);
                uint32_t occ = st & pair;
                if (occ == 0 || occ == pair) continue;
                uint32_t src = st ^ pair;                      // the electron sits on the other end
                int hopped = __builtin_popcount(st & between[b]);   // same count before and after the hop
                out.col[(size_t)k] = (int32_t)rank_of(src);
                out.plus[(size_t)k] = (uint8_t)(hopped & 1);   // -t * (-1)^hopped
                ++k;
            }
        }
    } catch (const std::bad_alloc &) {
        return -2;
    }
    return 0;
}

void canonical_ell(const SpinTable &tab, double t, int *width_out, int32_t *cols, double *vals)
{
    struct E { int32_t c; double v; };
    std::vector<E> row;
    // pass 1: merged width
    int width = 0;
    std::vector<int32_t> tmp;
    for (int64_t r = 0; r < tab.dim; ++r) {
        tmp.assign(tab.col.begin() + tab.rowptr[r], tab.col.begin() + tab.rowptr[r + 1]);
        std::sort(tmp.begin(), tmp.end());
        int n = (int)(std::unique(tmp.begin(), tmp.end()) - tmp.begin());
        if (t == 0.0) n = 0;
        width = std::max(width, n);
    }
    if (width_out) *width_out = width;
    if (!cols || !vals) return;
    for (int64_t r = 0; r < tab.dim; ++r) {
        row.clear();
        for (int64_t k = tab.rowptr[r]; k < tab.rowptr[r + 1]; ++k)
            row.push_back({tab.col[(size_t)k], tab.plus[(size_t)k] ? t : -t});
        std::stable_sort(row.begin(), row.end(), [](const E &a, const E &b) { return a.c < b.c; });
        int n = 0;
        for (size_t k = 0; k < row.size();) {
            int32_t c = row[k].c;
            double v = 0.0;
            while (k < row.size() && row[k].c == c) v += row[k++].v;
            if (v != 0.0) {
                cols[r * width + n] = c;
                vals[r * width + n] = v;
                ++n;
            }
        }
        for (; n < width; ++n) {
            cols[r * width + n] = -1;
            vals[r * width + n] = 0.0;
        }
    }
}

}  // namespace hub
