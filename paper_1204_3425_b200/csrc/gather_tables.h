// Host-side construction of the hop tables of variant GATHER (kernels_gather.cuh):
// batch-interleaved ELL over an INTERNAL order of the spin's basis states, with a
// shared-memory-bank-aware slot assignment and exact per-warp slot counts.
#pragma once
#include <cstdint>
#include <vector>

#include "host_tables.h"

namespace hub {

#ifndef GS_BATCH
#define GS_BATCH 8
#endif
constexpr int kSlotBatch = GS_BATCH;   // == kGatherBatch of the kernels

struct GatherTable {
    int64_t dim = 0;                // real states of the spin sector
    int64_t n_pos = 0;              // internal positions: dim rounded up to `align` (the tail is padding)
    int64_t ld = 0;                 // positions per batch plane (n_pos rounded up to 32)
    int w = 0;                      // slots per position in the table (multiple of kSlotBatch, >= every warp's count)
    std::vector<uint32_t> ent;      // [(k / 8) * ld + p] * 8 + k % 8 : target_position * 2 + neg
    std::vector<int32_t> cnt;       // per position: last slot holding a real entry + 1
    std::vector<uint16_t> wslots;   // per warp of 32 positions: slots EVERY lane of that warp walks (exact, not rounded)
    std::vector<int32_t> perm;      // position -> state index (ascending-bit-pattern order of PAPER.md:63-67), -1 = padding
    std::vector<int32_t> pos;       // state index -> position
    int64_t conflicts = 0;          // entries that share a bank with another lane of their wavefront
    int64_t wavefronts = 0;         // shared-memory wavefronts one tile costs: sum over warps of slots * 32 / lanes, + conflicts
    int symmetry_order = 0;         // order of the site-permutation group the internal order was built from (0: none)
    int64_t free_orbit_states = 0;  // states placed as whole orbits of that group
};

// `lanes` = lanes served by one shared-memory wavefront of the gather (128 bytes /
// bytes per staged element group: 8 for 16-byte groups, 16 for 8, 32 for 4); with
// lanes == 0 the entries keep the order of `tab` (no scheduling).  The zero slots
// of the staged tile (padding entries point at them) start at position n_pos =
// dim rounded up to `align` (the kernels pad a tile to one 128-byte line of pieces).
//
// sorted: the internal order is chosen for the gather (below); otherwise it is
// the basis order itself (perm = identity), which hubbard_apply's row-major
// vectors need.
//
// Internal order (sorted, lanes > 0).  If the bond list is given and the lattice
// has a group H of `lanes` site permutations that map the bond multiset onto
// itself (translations of a ring or torus, reflections; found by search), the
// states are grouped into ORBITS of H: the orbit {h_k s} of a state s occupies
// one aligned group of `lanes` positions, lane k holding h_k s.  All states of an
// orbit have the same number of hops (no padding inside a group), and the targets
// of slot j of the `lanes` lanes are again one whole orbit {h_k t_j} = `lanes`
// distinct lanes of another group: every bank carries exactly as many entries as
// a lane has hops, so the edge colouring places them without ANY bank conflict.
// Orbits are ordered by descending hop count (a warp's 4 groups are then nearly
// equal); the few states with a smaller orbit (invariant under some h) follow at
// the end.  Without such a group (or without a bond list) aligned groups of
// `lanes` consecutive basis states move as units, ordered by their longest row.
//
// Every lane of a warp walks the same number of slots W (wslots): a state's
// entries may therefore sit in ANY of its W slots.  For each group of `lanes`
// consecutive positions they are placed by a bipartite edge colouring (rows x
// banks) so that two entries of one slot do not hit the same bank.  W is chosen
// per warp to minimise its wavefronts: one more slot costs 32 / lanes wavefronts,
// one conflict costs one.
void build_gather_table(const SpinTable &tab, int lanes, int align, bool sorted, GatherTable &out,
                        const int32_t *bonds = nullptr, int n_bonds = 0);

}  // namespace hub
