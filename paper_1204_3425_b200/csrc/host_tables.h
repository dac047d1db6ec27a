// Host-side preparation: basis enumeration, ranks and per-spin
// hop lists.  Pure C++, no CUDA.  Product code: shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <vector>

namespace hub {

// One directed hop of one spin species: target row <- source column.
// sign_plus = true means the matrix element is +t, false means -t
// (element = -t * (-1)^{electrons hopped over}).
struct SpinTable {
    int n_sites = 0, n_el = 0;
    int64_t dim = 0;
    std::vector<uint32_t> states;      // ascending bit patterns
    // CSR over rows (row = state that receives amplitude), device-order entries:
    // duplicates (bond listed twice) are kept as separate entries.
    std::vector<int64_t> rowptr;       // dim + 1
    std::vector<int32_t> col;          // source state index
    std::vector<uint8_t> plus;         // 1: +t, 0: -t
    int width = 0;                     // max entries per row
};

// C(n, k) for 0 <= n <= 32 (fits in uint64).
uint64_t binom(int n, int k);

// Combinadic rank of a bit pattern among patterns with the same popcount
// (reading Q1 of DESIGN.md): sum_k C(p_k, k), p_1 < p_2 < ... the set bits.
int64_t rank_of(uint32_t s);

// Returns 0 on success, -1 invalid, -2 out of memory, -6 too large.
int build_spin_table(int n_sites, int n_el, const int32_t *bonds, int n_bonds, SpinTable &out);

// Canonical ELL (row-major dim x width, sorted by column, duplicates merged,
// zeros dropped, padding col=-1,val=0).  width_out = max nnz per row after
// merging.  cols/vals may be null to query the width only.
void canonical_ell(const SpinTable &tab, double t, int *width_out, int32_t *cols, double *vals);

}  // namespace hub
