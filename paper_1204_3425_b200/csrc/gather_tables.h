// Host-side construction of the hop tables of variant GATHER (kernels_gather.cuh):
// batch-interleaved ELL with a shared-memory-bank-aware slot assignment.
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
    int64_t ld = 0;                 // states per batch plane (dim rounded up to 32)
    int w = 0;                      // slots per state (multiple of kSlotBatch)
    std::vector<uint32_t> ent;      // [(k / 8) * ld + i] * 8 + k % 8 : col * 2 + neg
    std::vector<int32_t> cnt;       // per state: last used slot + 1
    int64_t conflicts = 0;          // entries that share a bank with another lane of their wavefront
};

// `lanes` = lanes served by one shared-memory wavefront of the gather
// (128 bytes / bytes per staged element group: 8 for 16-byte groups, 16 for 8,
// 32 for 4).  `zero_base` = index of the first of `lanes` zero slots of the
// staged tile (padding entries point at them).  With lanes == 0 the entries
// keep the order of `tab` (no scheduling).
//
// Within a warp every lane walks the same number of slots (the warp's longest
// row, rounded up to a batch), so a row's entries may sit in ANY of those
// slots.  For each group of `lanes` consecutive states the entries are placed
// by a bipartite edge colouring (rows x banks): two entries of one slot never
// hit the same bank unless the group has more entries on one bank than slots.
void build_gather_table(const SpinTable &tab, int lanes, int64_t zero_base, GatherTable &out);

}  // namespace hub
