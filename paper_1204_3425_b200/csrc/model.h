// Internal model state of libhubbard_b200 (not part of the ABI).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <vector>

#include "../../include/hubbard.h"
#include "host_tables.h"

namespace hub {

// Hop entry encoding shared by all device tables: e = col * 2 + plus,
// plus = 1 -> element +t, plus = 0 -> element -t.
// Padding entries of the down ELL point at the "zero slot" col = dim_dn.
constexpr uint32_t kPadEntry = 0xffffffffu;

// Device scalars of one Lanczos run; lives in device memory, written only by
// the finalising block of each sweep, read by every block of the next one.
struct LanczosScalars {
    double c_cur;    // f_j     = c_cur  * u_cur   (lazy normalisation)
    double c_prev;   // f_{j-1} = c_prev * u_prev
    double beta;     // b_j
    double alpha;    // a_j of the iteration in flight
    double amax;     // max_k |a_k| so far (breakdown rule, reading Q11)
    double tau;
    int j;           // iterations completed
    int stop;        // breakdown (or bad start vector): later sweeps are no-ops
    unsigned ticket; // arrival counter of the sweep in flight
    int started; // norm-producing sweeps finished (variant GATHER)
    double qnorm2;   // |q_j|^2 of the iteration in flight (variant GATHER, folded form: b_{j+1}^2 = |q_j|^2 - a_j^2 ahead of the ROW sweep)
};

// One spin's hop table in the device layout of variant GATHER (gather_tables.h): batch-interleaved ELL over the
// table's INTERNAL order of the basis states (position p <-> state perm[p]), entry = target_position * 2 + neg,
// the matrix element being t * (neg ? -1 : +1); padding entries are (n_pos + z) * 2 (the zero
// slots of the staged tile, sign +).
struct SpinDev {
    int64_t dim;            // dim_sigma (real states; positions >= dim are padding)
    int64_t n_pos;          // positions of a staged tile: dim rounded up to the tile height R
    int64_t ld;             // positions per batch plane (multiple of 32): entry k of position p
                            // sits at [((k / 8) * ld + p) * 8 + k % 8]
    int w;                  // slots per position in the table (multiple of 8)
    const uint16_t *e16;    // when n_pos + 128 <= 32768, else null: the entries in 16 bits - even slots as in e32,
                            // odd slots as target_position | neg << 15 (what the packed-word decode wants)
    const uint32_t *e32;    // entries (always present)
    const uint16_t *wslots; // per warp of 32 positions: slots every lane of that warp walks (exact)
    const int32_t *perm;    // position -> state index in the basis order of PAPER.md:63-67 (-1: padding)
    const uint32_t *st;     // basis bit patterns in position order (0 for padding)
};

// Everything a kernel needs to know about the model (passed by value).
struct DevModel {
    int64_t dim_up, dim_dn;
    const uint32_t *st_up, *st_dn;       // basis bit patterns
    // up table, row-major ELL [dim_up][w_up] (row-uniform access)
    const uint32_t *up_ent;
    const int32_t *up_cnt;
    int w_up;
    // down table, column-major ELL [w_dn][ld_dn] (coalesced over i_dn)
    const uint32_t *dn_ent32;
    const uint16_t *dn_ent16;            // compact copy when dim_dn + 1 <= 32768, else null
    const int32_t *dn_cnt;
    int w_dn;
    int64_t ld_dn;
    double t, U;
    SpinDev g_up, g_dn;                  // tables of variant GATHER in basis order (row-major callers: hubbard_apply)
    SpinDev gs_up, gs_dn;                // the same in the sorted internal order of the Lanczos work vectors
};

struct ProfRecord {
    int kclass;
    cudaEvent_t e0, e1;
};

// Development / test knobs, set per model with hubbard_debug_set (include/hubbard.h); the defaults are what
// bench.py times.  Nothing here is read from the environment.
struct DebugOptions {
    int gather_R = 0;               // cap on the tile height R of variant GATHER (0 = none)
    int gather_nosched = 0;         // 1: hop entries in bond order, no bank-aware placement
    int gather_nosort = 0;          // 1: the Lanczos work vectors keep the basis order (no internal reordering)
    int gather_nosymmetry = 0;      // 1: internal order from hop counts only (no lattice-symmetry orbits)
    int gather_ctas = 4;            // CTAs per SM for small tiles
    int gather_tmem_entries = 1;    // folded form: the COL sweep keeps the first hop-entry batch of its positions in tensor memory
    int gather_fold = 1;            // eight-pass Lanczos form (- b f_{j-1} folded into the ROW sweep through tensor memory):
                                    // 0 never, 1 where one tile fills the SM (automatic), 2 wherever the tensor memory suffices
    int apply_pure_gather = 0;      // 1: plain hubbard_apply as two gather sweeps instead of the hybrid
    int twosweep_old_row = 0;       // 1: TWOSWEEP fallback keeps the first row kernel
    int row_R = 0;                  // rows per CTA of the TWOSWEEP row kernel (0 = automatic)
    int strip_mb = 24;              // L2 budget of a column strip (MB)
    int strip_rb = 0;               // rows per block of the strip sweep (0 = automatic)
    int persist_max_dim = 1 << 17;  // largest dim AUTO runs in the cooperative kernel
    int force_cluster_row = 0;      // 1: take the path of rows larger than one SM
    int no_cluster_row = 0;         // 1: never use the cluster row sweep
    int cluster_R = 0, cluster_NC = 0;   // force one (R, NC) of the cluster row sweep
    int paper_subvectors = 1;       // variant PAPER: sub-vectors per block (1, or 4 = the paper's tuned form)
};

}  // namespace hub

struct hubbard_model {
    int n_sites = 0, n_up = 0, n_dn = 0, dtype = HUBBARD_F64;
    double t = 0, U = 0;
    std::vector<int32_t> bonds;
    hub::SpinTable up, dn;
    bool has_device = false;
    int variant = HUBBARD_VARIANT_AUTO;
    double tau = -1.0;                 // < 0: default for the dtype
    int last_cuda_error = 0;
    int64_t launches = 0;
    int sm_count = 148;
    int max_smem_optin = 0;
    int coop_launch = 0;               // device supports cooperative launches (variant PERSIST)
    int cluster_row = 0;               // rows go through clusters (kernels_cluster.cuh): gather_R == 0 but a cluster holds them
    int cluster_R = 0, cluster_NC = 0, cluster_part = 0;
    int gather_R = 0;                  // tile height of variant GATHER, 0 = does not fit
    int gather_symmetry = 0;           // order of the lattice symmetry group behind the internal order (0: none)
    hub::DebugOptions opt;
    std::vector<void *> layout_allocs;  // device tables that depend on `opt` (rebuilt by hubbard_debug_set)

    hub::DevModel dev{};
    std::vector<void *> dev_allocs;    // everything to cudaFree
    // Lanczos state (allocated on first use)
    void *work[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // 2 (PAPER/TWOSWEEP) or 5 (GATHER) in use, [5]: psi
    size_t work_bytes[6] = {0, 0, 0, 0, 0, 0};
    double *d_ycoef = nullptr;         // eigenvector of T_m for the ground-state pass
    int ycoef_cap = 0;
    hub::LanczosScalars *d_scal = nullptr;
    double *d_partial = nullptr;       // per-block partial sums
    int64_t n_partial = 0;
    double *d_alpha = nullptr, *d_beta = nullptr;
    int coef_cap = 0;
    // staging for the *_host entry points
    void *stage[2] = {nullptr, nullptr};
    // complex propagation: the same lattice with the up sector listed twice (real part ; imaginary part of a state
    // stacked as one real vector), and three device buffers of 2 * dim elements
    unsigned *shard_ticket = nullptr;   // arrival counter of the row-sharded vector kernels
    void *noalloc_scratch = nullptr;    // device address of the library's fixed scratch array on this model's GPU
                                        // (lanczos_shard_update_noalloc; resolved by hubbard_create, never allocated or freed)
    hubbard_model *twin = nullptr;
    void *cplx[3] = {nullptr, nullptr, nullptr};

    bool profiling = false;
    std::vector<hub::ProfRecord> prof;
    std::vector<cudaEvent_t> event_pool;   // reused by the profiling scopes
    int64_t prof_launches[HUBBARD_N_KCLASS] = {0};
    double prof_ms[HUBBARD_N_KCLASS] = {0};
};
