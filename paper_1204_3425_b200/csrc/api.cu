// C ABI of libhubbard_b200 (include/hubbard.h): model construction, table
// upload, kernel launches.  Nothing here throws across the boundary.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <unordered_map>

#include "kernels_cluster.cuh"
#include "kernels_gather.cuh"
#include "kernels_lanczos.cuh"
#include "kernels_paper.cuh"
#include "kernels_persist.cuh"
#include "kernels_twosweep.cuh"
#include "gather_tables.h"
#include "model.h"

using namespace hub;

namespace {

#define CU_TRY(m, expr)                                                   \
    do {                                                                  \
        cudaError_t e__ = (expr);                                         \
        if (e__ != cudaSuccess) {                                         \
            (m)->last_cuda_error = (int)e__;                              \
            cudaGetLastError();                                           \
            return (e__ == cudaErrorMemoryAllocation) ? HUBBARD_ERR_DEVICE_OOM : HUBBARD_ERR_CUDA; \
        }                                                                 \
    } while (0)

// `layout` = the table depends on the model's DebugOptions and is rebuilt when they change
template <typename U>
int dev_upload(hubbard_model *m, const std::vector<U> &h, const U **out, bool layout = false)
{
    void *p = nullptr;
    size_t bytes = std::max<size_t>(h.size(), 1) * sizeof(U);
    CU_TRY(m, cudaMalloc(&p, bytes));
    (layout ? m->layout_allocs : m->dev_allocs).push_back(p);
    if (!h.empty()) CU_TRY(m, cudaMemcpy(p, h.data(), h.size() * sizeof(U), cudaMemcpyHostToDevice));
    *out = static_cast<const U *>(p);
    return HUBBARD_OK;
}

size_t elem_size(const hubbard_model *m) { return m->dtype == HUBBARD_F32 ? 4 : 8; }
int64_t gather_align(const hubbard_model *m);
int64_t model_dim(const hubbard_model *m) { return m->up.dim * m->dn.dim; }

int build_host(hubbard_model **out, int n_sites, int n_up, int n_dn, const int32_t *bonds, int n_bonds,
               double t, double U, int dtype)
{
    if (!out) return HUBBARD_ERR_INVALID;
    *out = nullptr;
    if (dtype != HUBBARD_F32 && dtype != HUBBARD_F64) return HUBBARD_ERR_INVALID;
    if (!std::isfinite(t) || !std::isfinite(U)) return HUBBARD_ERR_INVALID;
    hubbard_model *m = new (std::nothrow) hubbard_model();
    if (!m) return HUBBARD_ERR_HOST_OOM;
    int rc = build_spin_table(n_sites, n_up, bonds, n_bonds, m->up);
    if (rc == 0) rc = build_spin_table(n_sites, n_dn, bonds, n_bonds, m->dn);
    if (rc != 0) {
        delete m;
        return rc == -1 ? HUBBARD_ERR_INVALID : rc == -2 ? HUBBARD_ERR_HOST_OOM : HUBBARD_ERR_UNSUPPORTED;
    }
    m->n_sites = n_sites; m->n_up = n_up; m->n_dn = n_dn; m->dtype = dtype; m->t = t; m->U = U;
    try {
        m->bonds.assign(bonds, bonds + 2 * (size_t)n_bonds);
    } catch (const std::bad_alloc &) {
        delete m;
        return HUBBARD_ERR_HOST_OOM;
    }
    *out = m;
    return HUBBARD_OK;
}

// Tile height R (rows per ROW tile = columns per COL tile) of variant GATHER:
// the largest R with R * sizeof(T) <= 16 for which a whole row AND a whole
// column of V fit in shared memory; 0 if even R = 1 does not fit.
int gather_R_for(const hubbard_model *m)
{
    const size_t es = m->dtype == HUBBARD_F32 ? 4 : 8;
    const size_t budget = (size_t)std::max(0, m->max_smem_optin - 1024);
    const int64_t n_in = std::max(m->dn.dim, m->up.dim);
    if (m->opt.force_cluster_row) return 0;                     // tests: take the path of rows larger than one SM
    const int forced = m->opt.gather_R;
    for (int R = (int)(16 / es); R >= 1; R >>= 1) {
        if (forced > 0 && R > forced) continue;
        // tile + zero slots + per-warp slot counts (2 bytes per 32 positions)
        // tile (positions padded to R) + zero slots + per-warp slot counts (2 bytes per 32 positions)
        if ((size_t)(n_in + R + 128 / (R * es)) * R * es + (size_t)(n_in + R + 32) / 32 * 2 + 16 <= budget) return R;
    }
    return 0;
}

// A V row does not fit one SM but R rows fit the distributed shared memory of an NC-CTA cluster
// (kernels_cluster.cuh).  Returns false if no (R, NC) does.
bool cluster_row_config(const hubbard_model *m, int *R_out, int *NC_out, int *part_out)
{
    if (m->opt.no_cluster_row || m->dn.dim < 64) return false;
    const int es = m->dtype == HUBBARD_F32 ? 4 : 8;
    const int r_force = m->opt.cluster_R, nc_force = m->opt.cluster_NC;
    // measured on C5 fp64: (R, NC) = (1, 2) 48.7 ms, (2, 4) 77.9 ms per sweep (the remote fraction and the 16-byte
    // DSMEM loads dominate), single-SM L2 gathers 54.2 ms: the smallest cluster first, then the tallest tile
    for (int NC : {2, 4}) {
        if (nc_force && NC != nc_force) continue;
        for (int R = 16 / es; R >= 1; R >>= 1) {
            if (r_force && R != r_force) continue;
            const int64_t part = ((m->dn.dim + NC - 1) / NC + 31) / 32 * 32;
            const size_t need = (size_t)(part + 128 / (R * es)) * R * es;
            if (need + 1024 <= (size_t)m->max_smem_optin && part * (NC - 1) < m->dn.dim) {
                if (R_out) *R_out = R;
                if (NC_out) *NC_out = NC;
                if (part_out) *part_out = (int)part;
                return true;
            }
        }
    }
    return false;
}

// Hop table of one spin for variant GATHER (kernels_gather.cuh, gather_tables.h).
// `align`: the tile's positions (and with them the zero slots padding entries point at) start at dim rounded up to it
int upload_gather_table(hubbard_model *m, const SpinTable &tab, int R, int align, bool sorted, SpinDev *out)
{
    SpinDev G{};
    const int es = m->dtype == HUBBARD_F32 ? 4 : 8;
    const int lanes = m->opt.gather_nosched ? 0 : 128 / (R * es);
    GatherTable T;
    const bool sym = sorted && !m->opt.gather_nosymmetry;
    build_gather_table(tab, lanes, align, sorted && !m->opt.gather_nosort, T, sym ? m->bonds.data() : nullptr,
                       sym ? (int)(m->bonds.size() / 2) : 0);
    if (sorted) m->gather_symmetry = T.symmetry_order;
    G.dim = tab.dim; G.n_pos = T.n_pos; G.ld = T.ld; G.w = T.w;
    int rc;
    if ((rc = dev_upload(m, T.ent, &G.e32, true))) return rc;
    if ((rc = dev_upload(m, T.wslots, &G.wslots, true))) return rc;
    if ((rc = dev_upload(m, T.perm, &G.perm, true))) return rc;
    std::vector<uint32_t> st((size_t)T.ld, 0u);
    for (int64_t p = 0; p < tab.dim; ++p) st[(size_t)p] = tab.states[(size_t)T.perm[(size_t)p]];
    if ((rc = dev_upload(m, st, &G.st, true))) return rc;
    G.e16 = nullptr;
    if (T.n_pos + 128 <= 32768) {
        std::vector<uint16_t> e16(T.ent.size());
        // device form of the 16-bit entries (kernels_gather.cuh, hop_lo / hop_hi): even slots position << 1 | neg,
        // odd slots position | neg << 15 (a slot's parity is its index's: batches are 8 entries)
        for (size_t i = 0; i < T.ent.size(); ++i) {
            const uint32_t pos = T.ent[i] >> 1, neg = T.ent[i] & 1u;
            e16[i] = (uint16_t)((i & 1) ? (pos | (neg << 15)) : ((pos << 1) | neg));
        }
        if ((rc = dev_upload(m, e16, &G.e16, true))) return rc;
    }
    *out = G;
    return HUBBARD_OK;
}

// The tables whose layout depends on the model's DebugOptions (tile height of variant GATHER, cluster row
// configuration); called by hubbard_create and again by hubbard_debug_set when such an option changes.
int upload_layout_tables(hubbard_model *m)
{
    DevModel &D = m->dev;
    for (void *p : m->layout_allocs) cudaFree(p);
    m->layout_allocs.clear();
    D.g_up = SpinDev{}; D.g_dn = SpinDev{}; D.gs_up = SpinDev{}; D.gs_dn = SpinDev{};
    m->cluster_row = 0; m->cluster_R = m->cluster_NC = m->cluster_part = 0;
    int rc;
    try {
        // variant GATHER: both spins column-major, entry = col * 2 + neg
        m->gather_R = gather_R_for(m);
        if (m->gather_R > 0) {
            const int al = (int)gather_align(m);
            if ((rc = upload_gather_table(m, m->up, m->gather_R, al, false, &D.g_up))) return rc;
            if ((rc = upload_gather_table(m, m->dn, m->gather_R, al, false, &D.g_dn))) return rc;
            if ((rc = upload_gather_table(m, m->up, m->gather_R, al, true, &D.gs_up))) return rc;
            if ((rc = upload_gather_table(m, m->dn, m->gather_R, al, true, &D.gs_dn))) return rc;
        } else if (cluster_row_config(m, &m->cluster_R, &m->cluster_NC, &m->cluster_part)) {
            // R rows fit the shared memory of a cluster: down-spin table in that layout for kernels_cluster.cuh
            if ((rc = upload_gather_table(m, m->dn, m->cluster_R, m->cluster_R, false, &D.g_dn))) return rc;
            m->cluster_row = 1;
        }
    } catch (const std::bad_alloc &) {
        return HUBBARD_ERR_HOST_OOM;
    }
    return HUBBARD_OK;
}

// Device layouts of the two hop tables (see model.h / DESIGN.md "data layout").
int upload_tables(hubbard_model *m)
{
    DevModel &D = m->dev;
    D.dim_up = m->up.dim; D.dim_dn = m->dn.dim; D.t = m->t; D.U = m->U;
    int rc;
    if ((rc = dev_upload(m, m->up.states, &D.st_up))) return rc;
    if ((rc = dev_upload(m, m->dn.states, &D.st_dn))) return rc;
    try {
        // up: row-major ELL
        D.w_up = std::max(m->up.width, 1);
        std::vector<uint32_t> ue((size_t)m->up.dim * D.w_up, kPadEntry);
        std::vector<int32_t> uc((size_t)m->up.dim);
        for (int64_t r = 0; r < m->up.dim; ++r) {
            int n = (int)(m->up.rowptr[r + 1] - m->up.rowptr[r]);
            uc[(size_t)r] = n;
            for (int k = 0; k < n; ++k) {
                size_t s = (size_t)(m->up.rowptr[r] + k);
                ue[(size_t)r * D.w_up + k] = (uint32_t)m->up.col[s] * 2u + m->up.plus[s];
            }
        }
        if ((rc = dev_upload(m, ue, &D.up_ent))) return rc;
        if ((rc = dev_upload(m, uc, &D.up_cnt))) return rc;
        // down: column-major ELL, padded with the zero slot col = dim_dn
        D.w_dn = std::max(m->dn.width, 1);
        D.ld_dn = (m->dn.dim + 31) / 32 * 32;
        const uint32_t pad = (uint32_t)m->dn.dim * 2u;
        std::vector<uint32_t> de((size_t)D.ld_dn * D.w_dn, pad);
        std::vector<int32_t> dc((size_t)m->dn.dim);
        for (int64_t r = 0; r < m->dn.dim; ++r) {
            int n = (int)(m->dn.rowptr[r + 1] - m->dn.rowptr[r]);
            dc[(size_t)r] = n;
            for (int k = 0; k < n; ++k) {
                size_t s = (size_t)(m->dn.rowptr[r] + k);
                de[(size_t)k * D.ld_dn + r] = (uint32_t)m->dn.col[s] * 2u + m->dn.plus[s];
            }
        }
        if ((rc = dev_upload(m, de, &D.dn_ent32))) return rc;
        if ((rc = dev_upload(m, dc, &D.dn_cnt))) return rc;
        D.dn_ent16 = nullptr;
        if (m->dn.dim + 1 <= 32768) {
            std::vector<uint16_t> d16(de.size());
            for (size_t i = 0; i < de.size(); ++i) d16[i] = (uint16_t)de[i];
            if ((rc = dev_upload(m, d16, &D.dn_ent16))) return rc;
        }
    } catch (const std::bad_alloc &) {
        return HUBBARD_ERR_HOST_OOM;
    }
    return upload_layout_tables(m);
}

}  // namespace

// ------------------------------------------------------------------ launches
namespace {

// Events come from a per-model pool (created once, reused): no cudaEventCreate inside a timed region after warm-up.
bool pool_event(hubbard_model *m, cudaEvent_t *e)
{
    if (!m->event_pool.empty()) { *e = m->event_pool.back(); m->event_pool.pop_back(); return true; }
    return cudaEventCreate(e) == cudaSuccess;
}

struct ProfScope {
    hubbard_model *m;
    cudaStream_t st;
    ProfRecord rec{};
    bool on;
    ProfScope(hubbard_model *m_, int kclass, cudaStream_t st_) : m(m_), st(st_), on(m_->profiling)
    {
        if (!on) return;
        rec.kclass = kclass;
        if (!pool_event(m, &rec.e0)) { on = false; return; }
        if (!pool_event(m, &rec.e1)) { m->event_pool.push_back(rec.e0); on = false; return; }
        cudaEventRecord(rec.e0, st);
    }
    ~ProfScope()
    {
        if (!on) return;
        cudaEventRecord(rec.e1, st);
        m->prof.push_back(rec);
    }
};

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is per function and process-wide: it is raised at most once
// per (kernel, size) and never lowered, so the launch path of a warmed-up model makes no attribute call.
template <typename K>
int ensure_smem(hubbard_model *m, K kern, size_t smem, bool carveout = false)
{
    static std::mutex mu;
    static std::unordered_map<const void *, size_t> granted;
    std::lock_guard<std::mutex> lock(mu);
    size_t &cur = granted[(const void *)kern];
    if (cur >= smem && cur > 0) return HUBBARD_OK;
    CU_TRY(m, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (carveout) CU_TRY(m, cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
    cur = smem;
    return HUBBARD_OK;
}

int after_launch(hubbard_model *m)
{
    ++m->launches;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        m->last_cuda_error = (int)e;
        return HUBBARD_ERR_CUDA;
    }
    return HUBBARD_OK;
}

int ensure_partials(hubbard_model *m, int64_t n)
{
    if (n <= m->n_partial) return HUBBARD_OK;
    if (m->d_partial) cudaFree(m->d_partial);
    m->d_partial = nullptr;
    m->n_partial = 0;
    CU_TRY(m, cudaMalloc((void **)&m->d_partial, (size_t)n * sizeof(double)));
    m->n_partial = n;
    return HUBBARD_OK;
}

int gather_R(const hubbard_model *m) { return m->gather_R; }

bool gather_fits(const hubbard_model *m) { return gather_R(m) > 0; }

int64_t round_up(int64_t n, int64_t r) { return (n + r - 1) / r * r; }

// elements of one work vector of variant GATHER (either tile-major layout)
// both dimensions of the tile-major work vectors are padded to the tile height R
int64_t gather_align(const hubbard_model *m) { return std::max(1, gather_R(m)); }

int64_t gather_vec_elems(const hubbard_model *m)
{
    return round_up(m->up.dim, gather_align(m)) * round_up(m->dn.dim, gather_align(m));
}

int resolve_variant(const hubbard_model *m)
{
    if (m->variant != HUBBARD_VARIANT_AUTO) return m->variant;
    // very small sectors (C1): the Lanczos loop is launch-latency bound -> one cooperative kernel (measured: C1 10.8 vs
    // 17.2 us per iteration; already C2, 854 k elements, is faster with the gather sweeps: 31.8 vs 39.3 us)
    if (m->up.dim * m->dn.dim <= (int64_t)m->opt.persist_max_dim && m->coop_launch) return HUBBARD_VARIANT_PERSIST;
    if (m->dn.dim < 512 || m->up.dim < 512) return HUBBARD_VARIANT_PAPER;
    // GATHER pays off when the R x R blocks it writes transposed are whole sectors (R * sizeof(T) = 16);
    // with a narrower tile (C5 fp32: R = 1) its strided writes are 4-byte pieces and TWOSWEEP is faster.
    const int es = m->dtype == HUBBARD_F32 ? 4 : 8;
    return (gather_R(m) * es == 16) ? HUBBARD_VARIANT_GATHER : HUBBARD_VARIANT_TWOSWEEP;
}

// ---- variant GATHER
// shared memory of a gather sweep: the staged tile + its zero slots, then the per-warp slot counts
size_t gather_smem_bytes(int64_t n_in_p, int R, size_t es)
{
    return (size_t)(n_in_p + 128 / (R * es)) * R * es + (size_t)(round_up(n_in_p, 32) / 32) * sizeof(uint16_t);
}

// Small sectors: several CTAs per SM (their staging and gather phases overlap one another); the 64-register
// kernels allow 1024 threads per SM in total.
void gather_launch_shape(const hubbard_model *m, size_t smem, int *per_sm, int *threads)
{
    int n = (int)std::min<size_t>(4, (size_t)(m->max_smem_optin - 2048) / (smem + 1024));
    n = std::max(1, std::min(n, m->opt.gather_ctas));
    *per_sm = n;
    *threads = std::max(32, kGatherMaxThreads / n / 32 * 32);
}

// Tensor-memory columns one CTA needs to keep one 16-byte item per thread and gather iteration of a sweep whose
// contracted dimension is n_in (a warp addresses a quarter of the 128 lanes), as the power of two >= 32 that
// tcgen05.alloc takes; 0 if the resident CTAs of an SM would need more than its 512 columns.
int gather_tmem_cols(const hubbard_model *m, int64_t n_in, int words)
{
    const int R = gather_R(m);
    const size_t es = m->dtype == HUBBARD_F32 ? 4 : 8;
    const int64_t n_in_p = round_up(n_in, gather_align(m));
    int per_sm, threads;
    gather_launch_shape(m, gather_smem_bytes(n_in_p, R, es), &per_sm, &threads);
    const int64_t n_it = (round_up(n_in_p, 32) + threads - 1) / threads;
    const int64_t need = (int64_t)((threads / 32 + 3) / 4) * n_it * words;
    int64_t cols = 32;
    while (cols < need) cols *= 2;
    return (cols * per_sm <= 512) ? (int)cols : 0;
}

// Folded Lanczos form of variant GATHER: columns the ROW sweep allocates to park its tile of u_j.  0: the nine-pass form
// (knob 0; knob 1 = automatic and several CTAs per SM; or not enough tensor memory).  Knob 2 folds wherever it fits.
int gather_fold_cols(const hubbard_model *m)
{
    const int R = gather_R(m);
    if (!m->opt.gather_fold || R == 0) return 0;
    const size_t es = m->dtype == HUBBARD_F32 ? 4 : 8;
    if (R * es != 16) return 0;          // full-width tiles only (what AUTO runs as GATHER; narrower ones are test geometry)
    // automatic: only where one tile fills the SM (C4).  Measured with the fold forced: C3 (2 CTAs per SM) no gain
    // (ROW + COL 0.376 ms either way), C2 (4 CTAs per SM, 4 tiles each) 10 % slower (the allocation is per launch).
    int per_sm, threads;
    gather_launch_shape(m, gather_smem_bytes(round_up(m->dn.dim, gather_align(m)), R, es), &per_sm, &threads);
    if (m->opt.gather_fold == 1 && per_sm != 1) return 0;
    return gather_tmem_cols(m, m->dn.dim, 4);
}

// Folded form, COL sweep: columns for the first hop-entry batch (16 bytes) of every position of the up table
int gather_ent_cols(const hubbard_model *m)
{
    if (gather_fold_cols(m) == 0 || !m->opt.gather_tmem_entries) return 0;
    return gather_tmem_cols(m, m->up.dim, 4);
}

template <typename T, int R, typename E, bool COL, bool LZ, bool FOLD>
int launch_gather_fold(hubbard_model *m, GatherArgs<T> A, cudaStream_t st)
{
    auto kern = gather_sweep_kernel<T, R, E, COL, LZ, FOLD>;
    A.du_p = round_up(A.dim_up, gather_align(m));
    A.dd_p = round_up(A.dim_dn, gather_align(m));
    const int64_t n_in_p = COL ? A.du_p : A.dd_p;
    const size_t smem = gather_smem_bytes(n_in_p, R, sizeof(T));
    if (int rc = ensure_smem(m, kern, smem, true)) return rc;
    const int64_t tiles = (COL ? A.dd_p : A.du_p) / R;
    int per_sm, threads;
    gather_launch_shape(m, smem, &per_sm, &threads);
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(tiles, (int64_t)m->sm_count * per_sm));
    {
        ProfScope ps(m, COL ? 2 : 1, st);
        kern<<<grid, threads, smem, st>>>(A);
    }
    return after_launch(m);
}

template <typename T, int R, typename E, bool COL, bool LZ>
int launch_gather_inst(hubbard_model *m, GatherArgs<T> A, cudaStream_t st)
{
    if constexpr (LZ && sizeof(E) == 2) {
        if (A.fold_cols > 0) return launch_gather_fold<T, R, E, COL, LZ, true>(m, A, st);
    }
    A.fold_cols = 0;
    return launch_gather_fold<T, R, E, COL, LZ, false>(m, A, st);
}

// LZ: the Lanczos sweeps work in the sorted internal order of BOTH spins; plain apply (row-major callers) in basis order.
template <typename T, bool COL, bool LZ>
int launch_gather(hubbard_model *m, GatherArgs<T> A, cudaStream_t st)
{
    const DevModel &D = m->dev;
    A.in = LZ ? (COL ? D.gs_up : D.gs_dn) : (COL ? D.g_up : D.g_dn);
    A.st_out = LZ ? D.gs_up.st : D.st_up;
    A.dim_up = D.dim_up; A.dim_dn = D.dim_dn; A.t = m->t; A.U = m->U;
    const int R = gather_R(m);
    if (R == 0) return HUBBARD_ERR_INVALID;
    if (LZ) {
        // (two partials per block: q.f and |q|^2 of the COL sweep)
        int rc = ensure_partials(m, (int64_t)m->sm_count * 8); if (rc) return rc;
        A.partials = m->d_partial;
        A.fold_cols = gather_fold_cols(m);
        A.ent_cols = COL ? gather_ent_cols(m) : 0;
    }
    if (!A.in.e16) {
        if constexpr (sizeof(T) == 4) {
            if (R == 1) return launch_gather_inst<T, 1, uint32_t, COL, LZ>(m, A, st);
        }
        return HUBBARD_ERR_INVALID;      // dim >= 32767 only ever fits at 4 bytes per state
    }
    if constexpr (sizeof(T) == 4) {
        if (R == 4) return launch_gather_inst<T, 4, uint16_t, COL, LZ>(m, A, st);
    }
    if (R >= 2) return launch_gather_inst<T, 2, uint16_t, COL, LZ>(m, A, st);
    return launch_gather_inst<T, 1, uint16_t, COL, LZ>(m, A, st);
}

template <typename T>
int launch_to_rt(hubbard_model *m, const T *x, T *rt, cudaStream_t st)
{
    const int R = gather_R(m);
    const int64_t du = m->up.dim, dd = m->dn.dim, du_p = round_up(du, gather_align(m)), dd_p = round_up(dd, gather_align(m));
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((int64_t)m->sm_count * 8, (du_p / R * dd_p + 255) / 256));
    const int32_t *pu = m->dev.gs_up.perm, *pd = m->dev.gs_dn.perm;
    if constexpr (sizeof(T) == 4) {
        if (R == 4) { to_rt_kernel<T, 4><<<grid, 256, 0, st>>>(x, rt, du, dd, du_p, dd_p, pu, pd); return after_launch(m); }
    }
    if (R == 2) { to_rt_kernel<T, 2><<<grid, 256, 0, st>>>(x, rt, du, dd, du_p, dd_p, pu, pd); return after_launch(m); }
    to_rt_kernel<T, 1><<<grid, 256, 0, st>>>(x, rt, du, dd, du_p, dd_p, pu, pd);
    return after_launch(m);
}

template <typename T>
int launch_from_rt(hubbard_model *m, const T *rt, T *x, cudaStream_t st)
{
    const int R = gather_R(m);
    const int64_t du = m->up.dim, dd = m->dn.dim, du_p = round_up(du, gather_align(m)), dd_p = round_up(dd, gather_align(m));
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((int64_t)m->sm_count * 8, (du_p / R * dd_p + 255) / 256));
    const int32_t *pu = m->dev.gs_up.perm, *pd = m->dev.gs_dn.perm;
    if constexpr (sizeof(T) == 4) {
        if (R == 4) { from_rt_kernel<T, 4><<<grid, 256, 0, st>>>(rt, x, du, dd, du_p, dd_p, pu, pd); return after_launch(m); }
    }
    if (R == 2) { from_rt_kernel<T, 2><<<grid, 256, 0, st>>>(rt, x, du, dd, du_p, dd_p, pu, pd); return after_launch(m); }
    from_rt_kernel<T, 1><<<grid, 256, 0, st>>>(rt, x, du, dd, du_p, dd_p, pu, pd);
    return after_launch(m);
}

int ensure_work(hubbard_model *m, int n_vec, size_t bytes)
{
    for (int i = 0; i < n_vec; ++i) {
        if (m->work[i] && m->work_bytes[i] >= bytes) continue;
        if (m->work[i]) cudaFree(m->work[i]);
        m->work[i] = nullptr;
        m->work_bytes[i] = 0;
        CU_TRY(m, cudaMalloc(&m->work[i], std::max<size_t>(bytes, 16)));
        m->work_bytes[i] = bytes;
    }
    return HUBBARD_OK;
}

// ---- variant PAPER
template <typename T, bool LZ>
int launch_paper(hubbard_model *m, const T *x, T *y, cudaStream_t st)
{
    const DevModel &D = m->dev;
    const int sub = m->opt.paper_subvectors == 4 ? 4 : 1;
    int64_t bps = (D.dim_dn + kPaperThreads - 1) / kPaperThreads;
    int64_t gy = std::min<int64_t>((D.dim_up + sub - 1) / sub, 65535);
    if (LZ) gy = std::max<int64_t>(1, std::min<int64_t>(gy, (1 << 16) / bps));
    if (bps > 0x7fffffff) return HUBBARD_ERR_UNSUPPORTED;
    SweepArgs<T> A{x, y, LZ ? m->d_scal : nullptr, m->d_partial};
    if (LZ) { int rc = ensure_partials(m, bps * gy); if (rc) return rc; A.partials = m->d_partial; }
    ProfScope ps(m, 0, st);
    const dim3 grid((unsigned)bps, (unsigned)gy);
    const size_t smem = (size_t)sub * D.w_up * 4;
    if (sub == 4) hv_paper_kernel<T, LZ, 4><<<grid, kPaperThreads, smem, st>>>(D, A);
    else hv_paper_kernel<T, LZ, 1><<<grid, kPaperThreads, smem, st>>>(D, A);
    return after_launch(m);
}

// ---- variant TWOSWEEP
template <typename T, typename E, int R, bool LZ>
int launch_row_staged(hubbard_model *m, const SweepArgs<T> &A, const E *ent, size_t smem, cudaStream_t st)
{
    auto kern = row_sweep_kernel<T, E, R, LZ>;
    if (int rc = ensure_smem(m, kern, smem)) return rc;
    int per_sm = std::max(1, std::min(2, (int)((size_t)m->max_smem_optin / (smem + 1024))));
    int64_t groups = (m->dev.dim_up + R - 1) / R;
    int grid = (int)std::min<int64_t>(groups, (int64_t)m->sm_count * per_sm);
    ProfScope ps(m, 1, st);
    kern<<<grid, kRowThreads, smem, st>>>(m->dev, A, ent);
    return after_launch(m);
}

template <typename T, typename E, bool LZ>
int launch_row(hubbard_model *m, const SweepArgs<T> &A, const E *ent, cudaStream_t st)
{
    const DevModel &D = m->dev;
    constexpr int N = 16 / sizeof(T);
    auto need = [&](int R) { return ((size_t)R * D.dim_dn + N) * sizeof(T); };
    int R = m->opt.row_R;
    if (R == 0) {
        // default: the largest R in {4,2,1} that still lets two CTAs share an SM, else R = 1
        R = 1;
        for (int r : {4, 2})
            if (need(r) + 1024 <= (size_t)m->max_smem_optin / 2) { R = r; break; }
    }
    if (R != 1 && R != 2 && R != 4) R = 1;
    while (R > 1 && need(R) > (size_t)m->max_smem_optin) R >>= 1;
    if (need(R) > (size_t)m->max_smem_optin) {
        int64_t bps = (D.dim_dn + kPaperThreads - 1) / kPaperThreads;
        int64_t gy = std::min<int64_t>(D.dim_up, 65535);
        ProfScope ps(m, 1, st);
        row_sweep_direct_kernel<T, E, LZ><<<dim3((unsigned)bps, (unsigned)gy), kPaperThreads, 0, st>>>(D, A, ent);
        return after_launch(m);
    }
    switch (R) {
        case 4: return launch_row_staged<T, E, 4, LZ>(m, A, ent, need(4), st);
        case 2: return launch_row_staged<T, E, 2, LZ>(m, A, ent, need(2), st);
        default: return launch_row_staged<T, E, 1, LZ>(m, A, ent, need(1), st);
    }
}

template <typename T, bool LZ>
int launch_strip(hubbard_model *m, SweepArgs<T> A, cudaStream_t st)
{
    const DevModel &D = m->dev;
    constexpr int N = 16 / sizeof(T);
    int VW = N;
    while (VW > 1 && (D.dim_dn % VW) != 0) VW >>= 1;
    StripPlan P;
    double mb = (double)m->opt.strip_mb;
    int64_t W = (int64_t)(mb * 1048576.0 / ((double)D.dim_up * sizeof(T)));
    W = std::max<int64_t>(32, W / 32 * 32);
    int64_t dd_up = (D.dim_dn + VW - 1) / VW * VW;
    W = std::min(W, dd_up);
    P.W = W;
    P.n_strips = (D.dim_dn + W - 1) / W;
    int RB = m->opt.strip_rb;
    if (RB <= 0) RB = (int)std::max<int64_t>(8, (2048 * (int64_t)VW + W - 1) / W);
    RB = (int)std::min<int64_t>(RB, D.dim_up);
    P.RB = RB;
    P.bps = (D.dim_up + RB - 1) / RB;
    int64_t nb = P.n_strips * P.bps;
    if (nb > 0x7fffffff) return HUBBARD_ERR_UNSUPPORTED;
    if (LZ) { int rc = ensure_partials(m, nb); if (rc) return rc; A.partials = m->d_partial; }
    size_t smem = (size_t)RB * (D.w_up + 1) * 4;
    ProfScope ps(m, 2, st);
    if (VW == 4) {
        if constexpr (sizeof(T) == 4) strip_sweep_kernel<T, 4, LZ><<<(unsigned)nb, kStripThreads, smem, st>>>(D, A, P);
    } else if (VW == 2) {
        strip_sweep_kernel<T, 2, LZ><<<(unsigned)nb, kStripThreads, smem, st>>>(D, A, P);
    } else {
        strip_sweep_kernel<T, 1, LZ><<<(unsigned)nb, kStripThreads, smem, st>>>(D, A, P);
    }
    return after_launch(m);
}

// Row half for rows larger than one SM's shared memory: clusters, the rows in distributed shared memory.
template <typename T, typename E, int R, int NC>
int launch_cluster_row_inst(hubbard_model *m, const ClusterRowArgs<T> &A, cudaStream_t st)
{
    auto kern = row_cluster_kernel<T, E, R, NC>;
    const size_t smem = (size_t)(A.part + 128 / (R * sizeof(T))) * R * sizeof(T);
    if (int rc = ensure_smem(m, kern, smem)) return rc;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)std::max(NC, m->sm_count / NC * NC));
    cfg.blockDim = dim3(kClusterThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr{};
    attr.id = cudaLaunchAttributeClusterDimension;
    attr.val.clusterDim.x = NC; attr.val.clusterDim.y = 1; attr.val.clusterDim.z = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
    ProfScope ps(m, 1, st);
    CU_TRY(m, cudaLaunchKernelEx(&cfg, kern, A));
    return after_launch(m);
}

template <typename T, typename E>
int launch_cluster_row_e(hubbard_model *m, const ClusterRowArgs<T> &A, cudaStream_t st)
{
    const int R = m->cluster_R, NC = m->cluster_NC;
    if constexpr (sizeof(T) == 4) {
        if (R == 4) return NC == 2 ? launch_cluster_row_inst<T, E, 4, 2>(m, A, st) : launch_cluster_row_inst<T, E, 4, 4>(m, A, st);
    }
    if (R == 2) return NC == 2 ? launch_cluster_row_inst<T, E, 2, 2>(m, A, st) : launch_cluster_row_inst<T, E, 2, 4>(m, A, st);
    return NC == 2 ? launch_cluster_row_inst<T, E, 1, 2>(m, A, st) : launch_cluster_row_inst<T, E, 1, 4>(m, A, st);
}

template <typename T>
int launch_cluster_row(hubbard_model *m, const T *x, T *y, LanczosScalars *S, cudaStream_t st)
{
    ClusterRowArgs<T> A{};
    A.in = m->dev.g_dn; A.st_up = m->dev.st_up; A.dim_up = m->dev.dim_up; A.dim_dn = m->dev.dim_dn;
    A.part = m->cluster_part;
    A.t = m->t; A.U = m->U; A.x = x; A.y = y; A.S = S;
    return A.in.e16 ? launch_cluster_row_e<T, uint16_t>(m, A, st) : launch_cluster_row_e<T, uint32_t>(m, A, st);
}

// y = H x (LZ = false) or the fused Lanczos H f_j - b_j f_{j-1}, a_j (LZ = true)
template <typename T, bool LZ>
int apply_impl(hubbard_model *m, const T *x, T *y, cudaStream_t st)
{
    m->dev.U = m->U;
    const int variant = resolve_variant(m);
    // PERSIST is a Lanczos-loop variant; its plain H v (and its classic fallback) is the PAPER kernel
    if (variant == HUBBARD_VARIANT_PAPER || variant == HUBBARD_VARIANT_PERSIST) return launch_paper<T, LZ>(m, x, y, st);
    if (variant == HUBBARD_VARIANT_GATHER) {
        if (LZ) return HUBBARD_ERR_INVALID;          // the Lanczos form of GATHER is lanczos_gather_impl
        if (m->variant == HUBBARD_VARIANT_AUTO && !m->opt.apply_pure_gather) {
            // plain y = H x on row-major vectors: gather ROW sweep (down term + diagonal, written row-major, no
            // intermediate layouts) followed by the strip sweep of TWOSWEEP (up term over L2-resident strips):
            // measured 4.0 ms against 5.0 ms for either pure form on C4 fp64
            GatherArgs<T> G{};
            G.x = x; G.y = y; G.y_rowmajor = 1;
            int rc = launch_gather<T, false, false>(m, G, st);
            if (rc) return rc;
            SweepArgs<T> A{x, y, nullptr, m->d_partial};
            return launch_strip<T, false>(m, A, st);
        }
        // two internal CT-layout vectors: x and z = (t H_dn + D) x
        int rc = ensure_work(m, 2, (size_t)gather_vec_elems(m) * sizeof(T));
        if (rc) return rc;
        GatherArgs<T> G{};
        G.x = x; G.y = y;
        G.Wct = static_cast<T *>(m->work[0]); G.Zct = static_cast<T *>(m->work[1]);
        if ((rc = launch_gather<T, false, false>(m, G, st))) return rc;
        return launch_gather<T, true, false>(m, G, st);
    }
    SweepArgs<T> A{x, y, LZ ? m->d_scal : nullptr, m->d_partial};
    int rc;
    if (m->variant == HUBBARD_VARIANT_AUTO && gather_R(m) > 0 && !m->opt.twosweep_old_row) {
        // AUTO fell back to TWOSWEEP because the tile is narrower than 16 bytes (C5 fp32): the row half still runs
        // as the gather ROW sweep on row-major vectors (batch-interleaved, bank-aware tables; vectorised staging)
        GatherArgs<T> G{};
        G.x = x; G.y = y; G.y_rowmajor = 1; G.S = LZ ? m->d_scal : nullptr;
        rc = launch_gather<T, false, false>(m, G, st);
    } else if (m->variant == HUBBARD_VARIANT_AUTO && m->cluster_row && (LZ || m->opt.force_cluster_row)) {
        // (plain apply, which reads no y, is faster through the single-SM L2 gathers: 39.6 vs 47 ms on C5 fp64)
        rc = launch_cluster_row<T>(m, x, y, LZ ? m->d_scal : nullptr, st);
    } else {
        rc = m->dev.dn_ent16 ? launch_row<T, uint16_t, LZ>(m, A, m->dev.dn_ent16, st)
                             : launch_row<T, uint32_t, LZ>(m, A, m->dev.dn_ent32, st);
    }
    if (rc) return rc;
    return launch_strip<T, LZ>(m, A, st);
}

}  // namespace

// --------------------------------------------------------------- Lanczos run
namespace {

int ensure_lanczos_state(hubbard_model *m, int iters, int n_vec)
{
    const size_t bytes = (size_t)(n_vec > 2 ? gather_vec_elems(m) : model_dim(m)) * elem_size(m);
    int rc0 = ensure_work(m, n_vec, bytes);
    if (rc0) return rc0;
    if (!m->d_scal) CU_TRY(m, cudaMalloc((void **)&m->d_scal, sizeof(LanczosScalars)));
    if (iters > m->coef_cap) {
        if (m->d_alpha) cudaFree(m->d_alpha);
        if (m->d_beta) cudaFree(m->d_beta);
        m->d_alpha = m->d_beta = nullptr;
        m->coef_cap = 0;
        CU_TRY(m, cudaMalloc((void **)&m->d_alpha, (size_t)iters * sizeof(double)));
        CU_TRY(m, cudaMalloc((void **)&m->d_beta, (size_t)iters * sizeof(double)));
        m->coef_cap = iters;
    }
    return HUBBARD_OK;
}

int fetch_coefficients(hubbard_model *m, int iters, double *alpha, double *beta, int *done, cudaStream_t st)
{
    LanczosScalars h{};
    CU_TRY(m, cudaMemcpyAsync(&h, m->d_scal, sizeof(h), cudaMemcpyDeviceToHost, st));
    CU_TRY(m, cudaStreamSynchronize(st));
    int n = std::max(0, std::min(h.j, iters));
    if (n > 0) {
        CU_TRY(m, cudaMemcpy(alpha, m->d_alpha, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost));
        CU_TRY(m, cudaMemcpy(beta, m->d_beta, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost));
    }
    if (done) *done = n;
    return HUBBARD_OK;
}

// What one call of the Lanczos engine does: iterations [j0, j1) of Algorithm 1,
// optionally the start (copy of v0, scalars) and the closing norm; with `ycoef`
// it also accumulates psi += y_j f_j (second pass for the ground-state vector).
struct LanczosPlan {
    int j0 = 0, j1 = 0;
    bool init = true, finish = true;
    const double *ycoef = nullptr;   // device, y_1..y_m of T_m's eigenvector
    void *psi = nullptr;             // device, same layout as the engine's vectors
};

int lanczos_vec_grid(const hubbard_model *m, int64_t n)
{
    return (int)std::max<int64_t>(1, std::min<int64_t>((int64_t)m->sm_count * 4, (n + 2047) / 2048));
}

double lanczos_tau(const hubbard_model *m) { return m->tau >= 0 ? m->tau : (m->dtype == HUBBARD_F64 ? 1e-10 : 1e-5); }

// Variant GATHER: two sweeps per iteration, vector updates folded in
// (kernels_gather.cuh), one closing norm sweep for b_{m+1}.  Five work vectors:
// A, B in the RT layout (q / u, swapped every iteration), two w buffers in the CT
// layout (this iteration's w and the previous one = u_j) and z in CT.
template <typename T>
int lanczos_gather_steps(hubbard_model *m, const T *v0, const LanczosPlan &P, cudaStream_t st)
{
    int rc;
    const int64_t n_p = gather_vec_elems(m);
    const int vec_grid = lanczos_vec_grid(m, n_p);
    if ((rc = ensure_partials(m, std::max<int64_t>(vec_grid, (int64_t)m->sm_count * 8)))) return rc;
    T *rt[2] = {static_cast<T *>(m->work[0]), static_cast<T *>(m->work[1])};
    T *wct[2] = {static_cast<T *>(m->work[2]), static_cast<T *>(m->work[3])};
    T *zct = static_cast<T *>(m->work[4]);
    if (P.init) {
        ProfScope ps(m, 5, st);
        if ((rc = launch_to_rt<T>(m, v0, rt[0], st))) return rc;                                    // "q_0" = f_1 unnormalised
        CU_TRY(m, cudaMemsetAsync(rt[1], 0, (size_t)n_p * sizeof(T), st));                          // line 2: f_0 <- 0
        CU_TRY(m, cudaMemsetAsync(wct[1], 0, (size_t)n_p * sizeof(T), st));
        if (P.psi) CU_TRY(m, cudaMemsetAsync(P.psi, 0, (size_t)n_p * sizeof(T), st));
        lanczos_scalars_init_kernel<<<1, 1, 0, st>>>(m->d_scal, lanczos_tau(m));                    // line 1: b_1 <- 0
        if ((rc = after_launch(m))) return rc;
    }
    GatherArgs<T> G{};
    G.S = m->d_scal; G.Zct = zct; G.alpha_out = m->d_alpha; G.beta_out = m->d_beta;
    for (int j = P.j0; j < P.j1; ++j) {
        G.Qrt = rt[j & 1]; G.Frt = rt[(j + 1) & 1]; G.Wct = wct[j & 1]; G.Fct = wct[(j + 1) & 1];
        if ((rc = launch_gather<T, false, true>(m, G, st))) return rc;     // lines 6-11 of j-1, row half of line 4
        if (P.psi) {                                                       // f_{j+1} = c w is complete: psi += y_{j+1} f_{j+1}
            psi_axpy_kernel<T><<<vec_grid, kVecThreads, 0, st>>>(static_cast<T *>(P.psi), G.Qrt, n_p, P.ycoef + j, m->d_scal);
            if ((rc = after_launch(m))) return rc;
        }
        if ((rc = launch_gather<T, true, true>(m, G, st))) return rc;      // line 4 (+ eq. 13), line 5
    }
    if (P.finish) {
        ProfScope ps(m, 3, st);
        lanczos_final_norm_kernel<T><<<vec_grid, 512, 0, st>>>(rt[P.j1 & 1], rt[(P.j1 + 1) & 1], n_p, m->d_scal, m->d_partial,
                                                               m->d_alpha, m->d_beta);
        if ((rc = after_launch(m))) return rc;
    }
    return HUBBARD_OK;
}

// Variants PAPER / TWOSWEEP: fused H f_j - b_j f_{j-1} with a_j, then the
// axpy + norm sweep (kernels_lanczos.cuh); two row-major work vectors.
template <typename T>
int lanczos_classic_steps(hubbard_model *m, const T *v0, const LanczosPlan &P, cudaStream_t st)
{
    int rc;
    const int64_t dim = model_dim(m);
    const int vec_grid = lanczos_vec_grid(m, dim);
    if ((rc = ensure_partials(m, vec_grid))) return rc;
    T *vec[2] = {static_cast<T *>(m->work[0]), static_cast<T *>(m->work[1])};
    if (P.init) {
        ProfScope ps(m, 5, st);
        CU_TRY(m, cudaMemcpyAsync(vec[0], v0, (size_t)dim * sizeof(T), cudaMemcpyDeviceToDevice, st));
        CU_TRY(m, cudaMemsetAsync(vec[1], 0, (size_t)dim * sizeof(T), st));   // line 2: f_0 <- 0
        if (P.psi) CU_TRY(m, cudaMemsetAsync(P.psi, 0, (size_t)dim * sizeof(T), st));
        CU_TRY(m, cudaMemsetAsync(m->d_scal, 0, sizeof(LanczosScalars), st));
        lanczos_init_kernel<T><<<vec_grid, kVecThreads, 0, st>>>(vec[0], dim, m->d_scal, m->d_partial, lanczos_tau(m));
        if ((rc = after_launch(m))) return rc;
    }
    for (int j = P.j0; j < P.j1; ++j) {
        T *cur = vec[j & 1], *prev = vec[(j + 1) & 1];
        if (P.psi) {                                                      // f_{j+1} = c_cur * cur
            psi_axpy_kernel<T><<<vec_grid, kVecThreads, 0, st>>>(static_cast<T *>(P.psi), cur, dim, P.ycoef + j, m->d_scal);
            if ((rc = after_launch(m))) return rc;
        }
        if ((rc = apply_impl<T, true>(m, cur, prev, st))) return rc;     // lines 4-5 (+ eq. 13)
        if ((rc = ensure_partials(m, vec_grid))) return rc;
        {
            ProfScope ps(m, 3, st);
            lanczos_axpy_norm_kernel<T><<<vec_grid, kVecThreads, 0, st>>>(cur, prev, dim, m->d_scal, m->d_partial,
                                                                         m->d_alpha, m->d_beta);   // lines 6-11
            if ((rc = after_launch(m))) return rc;
        }
    }
    return HUBBARD_OK;
}

// Variant PERSIST: the classic start, then ONE cooperative launch for all of [j0, j1) (kernels_persist.cuh).
template <typename T>
int lanczos_persist_steps(hubbard_model *m, const T *v0, const LanczosPlan &P, cudaStream_t st)
{
    int rc;
    const int64_t dim = model_dim(m);
    if (P.init) {
        LanczosPlan I = P;
        I.j0 = I.j1 = 0;
        if ((rc = lanczos_classic_steps<T>(m, v0, I, st))) return rc;          // copy of v0, f_0 = 0, c_1 = 1 / |v0|
    }
    if (P.j1 <= P.j0) return HUBBARD_OK;
    auto kern = lanczos_persistent_kernel<T>;
    int per_sm = 0;
    CU_TRY(m, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kPersistThreads, 0));
    if (per_sm < 1) return HUBBARD_ERR_CUDA;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((int64_t)m->sm_count * std::min(per_sm, 2),
                                                                  (dim + kPersistThreads - 1) / kPersistThreads));
    if ((rc = ensure_partials(m, std::max<int64_t>(2 * (int64_t)grid, lanczos_vec_grid(m, dim))))) return rc;
    m->dev.U = m->U;
    DevModel D = m->dev;
    PersistArgs<T> A{};
    A.vec0 = static_cast<T *>(m->work[0]); A.vec1 = static_cast<T *>(m->work[1]);
    A.S = m->d_scal; A.part_a = m->d_partial; A.part_b = m->d_partial + grid;
    A.alpha_out = m->d_alpha; A.beta_out = m->d_beta;
    A.j0 = P.j0; A.j1 = P.j1; A.ycoef = P.ycoef; A.psi = static_cast<T *>(P.psi);
    void *args[] = {&D, &A};
    {
        ProfScope ps(m, 0, st);
        CU_TRY(m, cudaLaunchCooperativeKernel((void *)kern, dim3(grid), dim3(kPersistThreads), args, 0, st));
    }
    return after_launch(m);
}

template <typename T>
int lanczos_steps(hubbard_model *m, const T *v0, const LanczosPlan &P, int coef_capacity, cudaStream_t st)
{
    const int variant = resolve_variant(m);
    const bool gather = variant == HUBBARD_VARIANT_GATHER;
    int rc = ensure_lanczos_state(m, coef_capacity, gather ? 5 : 2);
    if (rc) return rc;
    if (gather) return lanczos_gather_steps<T>(m, v0, P, st);
    if (variant == HUBBARD_VARIANT_PERSIST && m->coop_launch) return lanczos_persist_steps<T>(m, v0, P, st);
    return lanczos_classic_steps<T>(m, v0, P, st);
}

template <typename T>
int lanczos_impl(hubbard_model *m, const T *v0, int iters, double *alpha, double *beta, int *done, cudaStream_t st)
{
    LanczosPlan P;
    P.j1 = iters;
    int rc = lanczos_steps<T>(m, v0, P, iters, st);
    if (rc) return rc;
    return fetch_coefficients(m, iters, alpha, beta, done, st);
}

// Convergence-driven stopping ("the convergence of the ground state energy can be checked after
// each iteration"): every `check_every` iterations the coefficients so far are brought to the host and
// E_0^(m) = lambda_min(T_m) is compared with its previous value.
template <typename T>
int lanczos_until_impl(hubbard_model *m, const T *v0, int max_iters, int check_every, double tol, double *alpha,
                       double *beta, int *done, double *e0, cudaStream_t st)
{
    const bool gather = resolve_variant(m) == HUBBARD_VARIANT_GATHER;
    double e_prev = 0.0, e_cur = 0.0;
    bool have_prev = false, stopped = false;
    int j = 0;
    while (j < max_iters && !stopped) {
        LanczosPlan P;
        P.j0 = j; P.j1 = std::min(max_iters, j + check_every);
        P.init = (j == 0); P.finish = false;
        int rc = lanczos_steps<T>(m, v0, P, max_iters, st);
        if (rc) return rc;
        j = P.j1;
        // T_j needs a_1..a_j and b_2..b_j.  GATHER has recorded j-1 pairs and holds a_j in the scalars (b_{j+1}
        // comes with the next row sweep or the closing norm); the classic loop has recorded j pairs.
        LanczosScalars h{};
        CU_TRY(m, cudaMemcpyAsync(&h, m->d_scal, sizeof(h), cudaMemcpyDeviceToHost, st));
        CU_TRY(m, cudaStreamSynchronize(st));
        int n_rec = std::max(0, std::min(h.j, j));
        if (n_rec > 0) {
            CU_TRY(m, cudaMemcpy(alpha, m->d_alpha, (size_t)n_rec * sizeof(double), cudaMemcpyDeviceToHost));
            CU_TRY(m, cudaMemcpy(beta, m->d_beta, (size_t)n_rec * sizeof(double), cudaMemcpyDeviceToHost));
        }
        int mm = n_rec;
        if (h.stop) {
            stopped = true;                                  // breakdown (Algorithm 1 lines 8-10)
        } else if (gather && n_rec == j - 1) {
            alpha[n_rec] = h.alpha;
            mm = j;
        }
        if (mm >= 1) {
            if (lanczos_ground_energy(alpha, beta, mm, &e_cur) != HUBBARD_OK) return HUBBARD_ERR_INVALID;
            if (have_prev && std::fabs(e_cur - e_prev) <= tol * std::fmax(1.0, std::fabs(e_cur))) stopped = true;
            e_prev = e_cur;
            have_prev = true;
        }
    }
    {
        LanczosPlan P;
        P.j0 = P.j1 = j; P.init = false; P.finish = gather;   // closing norm: b_{m+1} for the last iteration
        int rc = lanczos_steps<T>(m, v0, P, max_iters, st);
        if (rc) return rc;
    }
    int n = 0;
    int rc = fetch_coefficients(m, max_iters, alpha, beta, &n, st);
    if (rc) return rc;
    if (done) *done = n;
    if (e0) {
        *e0 = e_cur;
        if (n >= 1) lanczos_ground_energy(alpha, beta, n, e0);
    }
    return HUBBARD_OK;
}

// Second Lanczos pass: out = sum_j y_j f_j (row-major, not normalised) for host coefficients y[0..n).  The run
// is bit-identical to the one that produced T_n (every reduction is deterministic), so the f_j are the same.
template <typename T>
int lanczos_combine(hubbard_model *m, const T *v0, int n, const double *y_host, T *out, cudaStream_t st)
{
    const bool gather = resolve_variant(m) == HUBBARD_VARIANT_GATHER;
    const int64_t n_vec = gather ? gather_vec_elems(m) : model_dim(m);
    int rc = ensure_work(m, gather ? 6 : 2, (size_t)n_vec * sizeof(T));
    if (rc) return rc;
    if (n > m->ycoef_cap) {
        if (m->d_ycoef) cudaFree(m->d_ycoef);
        m->d_ycoef = nullptr; m->ycoef_cap = 0;
        CU_TRY(m, cudaMalloc((void **)&m->d_ycoef, (size_t)n * sizeof(double)));
        m->ycoef_cap = n;
    }
    CU_TRY(m, cudaMemcpyAsync(m->d_ycoef, y_host, (size_t)n * sizeof(double), cudaMemcpyHostToDevice, st));
    LanczosPlan P;
    P.j1 = n; P.finish = false; P.ycoef = m->d_ycoef;
    // GATHER accumulates in its RT layout (work[5]) and converts at the end; the other loops are row-major already
    P.psi = gather ? m->work[5] : static_cast<void *>(out);
    if ((rc = lanczos_steps<T>(m, v0, P, n, st))) return rc;
    if (gather && (rc = launch_from_rt<T>(m, static_cast<const T *>(m->work[5]), out, st))) return rc;
    CU_TRY(m, cudaStreamSynchronize(st));      // y_host may go out of scope in the caller
    return HUBBARD_OK;
}

// Ground-state vector: pass 1 = the Lanczos run, host = eigenvector y of T_m, pass 2 = combine.
template <typename T>
int lanczos_ground_state_impl(hubbard_model *m, const T *v0, int iters, T *psi_out, double *e0, int *done, cudaStream_t st)
{
    std::vector<double> alpha((size_t)std::max(iters, 1)), beta((size_t)std::max(iters, 1)), y((size_t)std::max(iters, 1));
    int n = 0;
    int rc = lanczos_impl<T>(m, v0, iters, alpha.data(), beta.data(), &n, st);
    if (rc) return rc;
    if (done) *done = n;
    if (n < 1) return HUBBARD_ERR_INVALID;
    double lam = 0.0;
    if ((rc = lanczos_ground_vector(alpha.data(), beta.data(), n, &lam, y.data()))) return rc;
    if (e0) *e0 = lam;
    if ((rc = lanczos_combine<T>(m, v0, n, y.data(), psi_out, st))) return rc;
    const int64_t dim = model_dim(m);
    const int vec_grid = lanczos_vec_grid(m, dim);
    if ((rc = ensure_partials(m, vec_grid))) return rc;
    vec_norm2_kernel<T><<<vec_grid, kVecThreads, 0, st>>>(psi_out, dim, m->d_scal, m->d_partial);
    if ((rc = after_launch(m))) return rc;
    vec_normalise_kernel<T><<<vec_grid, kVecThreads, 0, st>>>(psi_out, dim, m->d_scal);
    if ((rc = after_launch(m))) return rc;
    CU_TRY(m, cudaStreamSynchronize(st));
    return HUBBARD_OK;
}

// Krylov propagation: exp(-(tau + i t) H) v0 ~ |v0| V_m exp(-(tau + i t) T_m) e_1 for a
// REAL start vector; the real and the imaginary part are each one combine pass.
template <typename T>
int lanczos_propagate_impl(hubbard_model *m, const T *v0, int iters, double tau, double t, T *out_re, T *out_im, int *done,
                           cudaStream_t st)
{
    std::vector<double> alpha((size_t)iters), beta((size_t)iters), yr((size_t)iters), yi((size_t)iters);
    int n = 0;
    int rc = lanczos_impl<T>(m, v0, iters, alpha.data(), beta.data(), &n, st);
    if (rc) return rc;
    if (done) *done = n;
    if (n < 1) return HUBBARD_ERR_INVALID;
    // |v0| (the run normalises its copy of v0 by a scalar; the propagated vector carries the norm)
    const int64_t dim = model_dim(m);
    const int vec_grid = lanczos_vec_grid(m, dim);
    if ((rc = ensure_partials(m, vec_grid))) return rc;
    vec_norm2_kernel<T><<<vec_grid, kVecThreads, 0, st>>>(v0, dim, m->d_scal, m->d_partial);
    if ((rc = after_launch(m))) return rc;
    LanczosScalars h{};
    CU_TRY(m, cudaMemcpyAsync(&h, m->d_scal, sizeof(h), cudaMemcpyDeviceToHost, st));
    CU_TRY(m, cudaStreamSynchronize(st));
    const double nrm = std::sqrt(h.beta);
    if ((rc = lanczos_expm_e1(alpha.data(), beta.data(), n, tau, t, yr.data(), yi.data()))) return rc;
    for (int j = 0; j < n; ++j) { yr[(size_t)j] *= nrm; yi[(size_t)j] *= nrm; }
    if ((rc = lanczos_combine<T>(m, v0, n, yr.data(), out_re, st))) return rc;
    if (out_im && (rc = lanczos_combine<T>(m, v0, n, yi.data(), out_im, st))) return rc;
    return HUBBARD_OK;
}

// ---- complex start vectors (second half): a propagated state is complex, psi = x + i y.  H is real
// symmetric, so Lanczos on psi is REAL Lanczos on the stacked vector [x ; y] with the block-diagonal operator
// diag(H, H) and the real inner product (the recurrence polynomials have real coefficients a_j, b_j, and
// <p(H) psi, q(H) psi> is real for real polynomials).  diag(H, H) is this library's H for the same lattice with the
// up sector listed twice: V becomes a (2 dim_up) x dim_dn matrix, H_up -> I_2 (x) H_up, the diagonal repeats.  The
// "twin" model holds exactly that and runs through the unchanged kernels.
int ensure_twin(hubbard_model *m)
{
    if (!m->twin) {
        hubbard_model *t = new (std::nothrow) hubbard_model();
        if (!t) return HUBBARD_ERR_HOST_OOM;
        try {
            t->n_sites = m->n_sites; t->n_up = m->n_up; t->n_dn = m->n_dn; t->dtype = m->dtype; t->t = m->t; t->U = m->U;
            t->bonds = m->bonds;
            t->dn = m->dn;
            const SpinTable &u = m->up;
            SpinTable &d = t->up;
            d.n_sites = u.n_sites; d.n_el = u.n_el; d.dim = 2 * u.dim; d.width = u.width;
            if (d.dim >= 0x7fffffffll) { delete t; return HUBBARD_ERR_UNSUPPORTED; }
            d.states = u.states;
            d.states.insert(d.states.end(), u.states.begin(), u.states.end());
            d.col = u.col;
            d.plus = u.plus;
            d.rowptr = u.rowptr;
            const int64_t nnz = u.rowptr[(size_t)u.dim];
            for (int64_t r = 1; r <= u.dim; ++r) d.rowptr.push_back(nnz + u.rowptr[(size_t)r]);
            for (int64_t k = 0; k < nnz; ++k) { d.col.push_back(u.col[(size_t)k] + (int32_t)u.dim); d.plus.push_back(u.plus[(size_t)k]); }
        } catch (const std::bad_alloc &) {
            delete t;
            return HUBBARD_ERR_HOST_OOM;
        }
        t->opt = m->opt;
        t->opt.gather_nosymmetry = 1;            // the orbit construction assumes distinct bit patterns
        t->sm_count = m->sm_count; t->max_smem_optin = m->max_smem_optin; t->coop_launch = m->coop_launch;
        int rc = upload_tables(t);
        if (rc) { hubbard_destroy(t); return rc; }
        t->has_device = true;
        m->twin = t;
    }
    hubbard_model *t = m->twin;
    t->U = m->U; t->dev.U = m->U; t->tau = m->tau;
    t->variant = (m->variant == HUBBARD_VARIANT_GATHER && !gather_fits(t)) ? HUBBARD_VARIANT_AUTO : m->variant;
    const size_t bytes = 2 * (size_t)model_dim(m) * elem_size(m);
    for (int k = 0; k < 3; ++k)
        if (!m->cplx[k]) CU_TRY(m, cudaMalloc(&m->cplx[k], std::max<size_t>(bytes, 16)));
    return HUBBARD_OK;
}

template <typename T>
int lanczos_propagate_complex_impl(hubbard_model *m, const T *re_in, const T *im_in, int iters, double tau, double t,
                                   T *out_re, T *out_im, int *done, cudaStream_t st)
{
    int rc = ensure_twin(m);
    if (rc) return rc;
    hubbard_model *tw = m->twin;
    const int64_t dim = model_dim(m);
    T *v2 = static_cast<T *>(m->cplx[0]), *A = static_cast<T *>(m->cplx[1]), *B = static_cast<T *>(m->cplx[2]);
    CU_TRY(m, cudaMemcpyAsync(v2, re_in, (size_t)dim * sizeof(T), cudaMemcpyDeviceToDevice, st));
    if (im_in) CU_TRY(m, cudaMemcpyAsync(v2 + dim, im_in, (size_t)dim * sizeof(T), cudaMemcpyDeviceToDevice, st));
    else CU_TRY(m, cudaMemsetAsync(v2 + dim, 0, (size_t)dim * sizeof(T), st));
    // real Lanczos on [x ; y] with diag(H, H): the existing real propagation gives A = Re-coefficients, B = Im-coefficients
    rc = lanczos_propagate_impl<T>(tw, v2, iters, tau, t, A, B, done, st);
    m->last_cuda_error = tw->last_cuda_error;
    m->launches += tw->launches; tw->launches = 0;
    if (rc) return rc;
    const int grid = lanczos_vec_grid(m, dim);
    complex_mix_kernel<T><<<grid, kVecThreads, 0, st>>>(A, B, dim, out_re, out_im);
    if ((rc = after_launch(m))) return rc;
    CU_TRY(m, cudaStreamSynchronize(st));
    return HUBBARD_OK;
}

int ensure_stage(hubbard_model *m, int which)
{
    if (m->stage[which]) return HUBBARD_OK;
    CU_TRY(m, cudaMalloc(&m->stage[which], std::max<size_t>((size_t)model_dim(m) * elem_size(m), 16)));
    return HUBBARD_OK;
}

// ---- fixed scratch of lanczos_shard_update_noalloc (include/hubbard.h): the arrival counter in the first 256 bytes,
// then one fp64 partial sum per block.  A file-scope device array: every GPU that loads this library holds these
// HUBBARD_NOALLOC_SCRATCH_BYTES until the process exits, and nobody ever allocates or frees them.  In HOST code the name
// `g_noalloc_scratch` is only a handle for the runtime, not a device address - a kernel given `g_noalloc_scratch`
// itself would fault (or, where the GPU can reach host memory, silently use the wrong memory): the address a kernel
// may be given comes from cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned char g_noalloc_scratch[HUBBARD_NOALLOC_SCRATCH_BYTES];

// Device address of g_noalloc_scratch on the CURRENT device (resolved on first use per device, then cached).
// Called at set-up (hubbard_create); allocates nothing.
int noalloc_scratch_for_current_device(hubbard_model *m, void **out)
{
    constexpr int kMaxDevices = 64;
    static std::mutex mu;
    static void *cached[kMaxDevices] = {nullptr};
    int dev = -1;
    CU_TRY(m, cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return HUBBARD_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(mu);
    if (!cached[dev]) {
        void *p = nullptr;
        CU_TRY(m, cudaGetSymbolAddress(&p, g_noalloc_scratch));
        cached[dev] = p;
    }
    *out = cached[dev];
    return HUBBARD_OK;
}

int check_device_model(const hubbard_model *m)
{
    if (!m) return HUBBARD_ERR_INVALID;
    if (!m->has_device) return HUBBARD_ERR_NO_DEVICE;
    return HUBBARD_OK;
}

}  // namespace

// ------------------------------------------------------------------ the ABI
extern "C" {

int hubbard_create_host(hubbard_model **out, int n_sites, int n_up, int n_dn, const int32_t *bonds, int n_bonds,
                        double t, double U, int dtype)
{
    return build_host(out, n_sites, n_up, n_dn, bonds, n_bonds, t, U, dtype);
}

int hubbard_create(hubbard_model **out, int n_sites, int n_up, int n_dn, const int32_t *bonds, int n_bonds,
                   double t, double U, int dtype)
{
    int rc = build_host(out, n_sites, n_up, n_dn, bonds, n_bonds, t, U, dtype);
    if (rc) return rc;
    hubbard_model *m = *out;
    auto fail = [&](int code) { hubbard_destroy(m); *out = nullptr; return code; };
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(HUBBARD_ERR_CUDA); }
    cudaDeviceGetAttribute(&m->sm_count, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&m->max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaDeviceGetAttribute(&m->coop_launch, cudaDevAttrCooperativeLaunch, dev);
    if (m->sm_count <= 0) m->sm_count = 148;
    rc = upload_tables(m);
    if (rc) return fail(rc);
    if ((rc = noalloc_scratch_for_current_device(m, &m->noalloc_scratch))) return fail(rc);
    m->has_device = true;
    return HUBBARD_OK;
}

void hubbard_destroy(hubbard_model *m)
{
    if (!m) return;
    for (auto &r : m->prof) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
    for (cudaEvent_t e : m->event_pool) cudaEventDestroy(e);
    for (void *p : m->dev_allocs) cudaFree(p);
    for (void *p : m->layout_allocs) cudaFree(p);
    for (int i = 0; i < 6; ++i) if (m->work[i]) cudaFree(m->work[i]);
    if (m->d_ycoef) cudaFree(m->d_ycoef);
    for (int i = 0; i < 2; ++i) if (m->stage[i]) cudaFree(m->stage[i]);
    for (int i = 0; i < 3; ++i) if (m->cplx[i]) cudaFree(m->cplx[i]);
    if (m->twin) hubbard_destroy(m->twin);
    if (m->shard_ticket) cudaFree(m->shard_ticket);
    if (m->d_scal) cudaFree(m->d_scal);
    if (m->d_partial) cudaFree(m->d_partial);
    if (m->d_alpha) cudaFree(m->d_alpha);
    if (m->d_beta) cudaFree(m->d_beta);
    delete m;
}

int hubbard_dims(const hubbard_model *m, int64_t *dim_up, int64_t *dim_dn)
{
    if (!m) return HUBBARD_ERR_INVALID;
    if (dim_up) *dim_up = m->up.dim;
    if (dim_dn) *dim_dn = m->dn.dim;
    return HUBBARD_OK;
}

int hubbard_set_U(hubbard_model *m, double U)
{
    if (!m || !std::isfinite(U)) return HUBBARD_ERR_INVALID;
    m->U = U;
    m->dev.U = U;
    return HUBBARD_OK;
}

int hubbard_set_variant(hubbard_model *m, int variant)
{
    if (!m || variant < HUBBARD_VARIANT_AUTO || variant > HUBBARD_VARIANT_PERSIST) return HUBBARD_ERR_INVALID;
    if (variant == HUBBARD_VARIANT_GATHER && m->has_device && !gather_fits(m)) return HUBBARD_ERR_INVALID;
    m->variant = variant;
    return HUBBARD_OK;
}

int lanczos_set_tau(hubbard_model *m, double tau)
{
    if (!m || !(tau >= 0.0)) return HUBBARD_ERR_INVALID;
    m->tau = tau;
    return HUBBARD_OK;
}

int hubbard_apply(hubbard_model *m, const void *x_dev, void *y_dev, void *stream)
{
    int rc = check_device_model(m);
    if (rc) return rc;
    if (!x_dev || !y_dev || x_dev == y_dev) return HUBBARD_ERR_INVALID;
    if (((uintptr_t)x_dev | (uintptr_t)y_dev) & 15) return HUBBARD_ERR_INVALID;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (m->dtype == HUBBARD_F32)
        return apply_impl<float, false>(m, static_cast<const float *>(x_dev), static_cast<float *>(y_dev), st);
    return apply_impl<double, false>(m, static_cast<const double *>(x_dev), static_cast<double *>(y_dev), st);
}

int lanczos_run(hubbard_model *m, const void *v0_dev, int iters, double *alpha_host, double *beta_host,
                int *iters_done, void *stream)
{
    int rc = check_device_model(m);
    if (rc) return rc;
    if (iters_done) *iters_done = 0;
    if (!v0_dev || iters < 0 || (iters > 0 && (!alpha_host || !beta_host))) return HUBBARD_ERR_INVALID;
    if ((uintptr_t)v0_dev & 15) return HUBBARD_ERR_INVALID;
    if (iters == 0) return HUBBARD_OK;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (m->dtype == HUBBARD_F32)
        return lanczos_impl<float>(m, static_cast<const float *>(v0_dev), iters, alpha_host, beta_host, iters_done, st);
    return lanczos_impl<double>(m, static_cast<const double *>(v0_dev), iters, alpha_host, beta_host, iters_done, st);
}

int lanczos_run_until(hubbard_model *m, const void *v0_dev, int max_iters, int check_every, double tol,
                      double *alpha_host, double *beta_host, int *iters_done, double *e0, void *stream)
{
    int rc = check_device_model(m);
    if (rc) return rc;
    if (iters_done) *iters_done = 0;
    if (!v0_dev || max_iters < 1 || check_every < 1 || !(tol >= 0.0) || !alpha_host || !beta_host) return HUBBARD_ERR_INVALID;
    if ((uintptr_t)v0_dev & 15) return HUBBARD_ERR_INVALID;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (m->dtype == HUBBARD_F32)
        return lanczos_until_impl<float>(m, static_cast<const float *>(v0_dev), max_iters, check_every, tol, alpha_host,
                                         beta_host, iters_done, e0, st);
    return lanczos_until_impl<double>(m, static_cast<const double *>(v0_dev), max_iters, check_every, tol, alpha_host,
                                      beta_host, iters_done, e0, st);
}

int lanczos_ground_state(hubbard_model *m, const void *v0_dev, int iters, void *psi_dev, double *e0, int *iters_done,
                         void *stream)
{
    int rc = check_device_model(m);
    if (rc) return rc;
    if (iters_done) *iters_done = 0;
    if (!v0_dev || !psi_dev || iters < 1 || v0_dev == psi_dev) return HUBBARD_ERR_INVALID;
    if (((uintptr_t)v0_dev | (uintptr_t)psi_dev) & 15) return HUBBARD_ERR_INVALID;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (m->dtype == HUBBARD_F32)
        return lanczos_ground_state_impl<float>(m, static_cast<const float *>(v0_dev), iters, static_cast<float *>(psi_dev), e0,
                                                iters_done, st);
    return lanczos_ground_state_impl<double>(m, static_cast<const double *>(v0_dev), iters, static_cast<double *>(psi_dev), e0,
                                             iters_done, st);
}

int lanczos_propagate(hubbard_model *m, const void *v0_dev, int iters, double tau, double t, void *out_re_dev,
                      void *out_im_dev, int *iters_done, void *stream)
{
    int rc = check_device_model(m);
    if (rc) return rc;
    if (iters_done) *iters_done = 0;
    if (!v0_dev || !out_re_dev || iters < 1 || !std::isfinite(tau) || !std::isfinite(t)) return HUBBARD_ERR_INVALID;
    if (v0_dev == out_re_dev || v0_dev == out_im_dev || out_re_dev == out_im_dev) return HUBBARD_ERR_INVALID;
    if (((uintptr_t)v0_dev | (uintptr_t)out_re_dev | (uintptr_t)out_im_dev) & 15) return HUBBARD_ERR_INVALID;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (m->dtype == HUBBARD_F32)
        return lanczos_propagate_impl<float>(m, static_cast<const float *>(v0_dev), iters, tau, t, static_cast<float *>(out_re_dev),
                                             static_cast<float *>(out_im_dev), iters_done, st);
    return lanczos_propagate_impl<double>(m, static_cast<const double *>(v0_dev), iters, tau, t, static_cast<double *>(out_re_dev),
                                          static_cast<double *>(out_im_dev), iters_done, st);
}

int lanczos_propagate_complex(hubbard_model *m, const void *re_in_dev, const void *im_in_dev, int iters, double tau, double t,
                              void *out_re_dev, void *out_im_dev, int *iters_done, void *stream)
{
    int rc = check_device_model(m);
    if (rc) return rc;
    if (iters_done) *iters_done = 0;
    if (!re_in_dev || !out_re_dev || !out_im_dev || iters < 1 || !std::isfinite(tau) || !std::isfinite(t)) return HUBBARD_ERR_INVALID;
    if (((uintptr_t)re_in_dev | (uintptr_t)im_in_dev | (uintptr_t)out_re_dev | (uintptr_t)out_im_dev) & 15) return HUBBARD_ERR_INVALID;
    if (out_re_dev == out_im_dev) return HUBBARD_ERR_INVALID;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (m->dtype == HUBBARD_F32)
        return lanczos_propagate_complex_impl<float>(m, static_cast<const float *>(re_in_dev), static_cast<const float *>(im_in_dev), iters,
                                                     tau, t, static_cast<float *>(out_re_dev), static_cast<float *>(out_im_dev), iters_done, st);
    return lanczos_propagate_complex_impl<double>(m, static_cast<const double *>(re_in_dev), static_cast<const double *>(im_in_dev), iters,
                                                  tau, t, static_cast<double *>(out_re_dev), static_cast<double *>(out_im_dev), iters_done, st);
}

// ---- row-sharded H v and Lanczos pieces
int hubbard_apply_rows(hubbard_model *m, const void *x_full_dev, void *y_rows_dev, int64_t row0, int64_t row1, void *stream)
{
    int rc = check_device_model(m);
    if (rc) return rc;
    if (!x_full_dev || !y_rows_dev || row0 < 0 || row1 < row0 || row1 > m->up.dim) return HUBBARD_ERR_INVALID;
    if (((uintptr_t)x_full_dev | (uintptr_t)y_rows_dev) & 15) return HUBBARD_ERR_INVALID;
    if (row1 == row0) return HUBBARD_OK;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    m->dev.U = m->U;
    const DevModel &D = m->dev;
    const int64_t bps = (D.dim_dn + kPaperThreads - 1) / kPaperThreads;
    if (bps > 0x7fffffff) return HUBBARD_ERR_UNSUPPORTED;
    const int64_t gy = std::min<int64_t>(row1 - row0, 65535);
    auto launch = [&](auto tag) {
        using T = decltype(tag);
        SweepArgs<T> A{static_cast<const T *>(x_full_dev), static_cast<T *>(y_rows_dev), nullptr, m->d_partial};
        A.a_begin = row0; A.a_end = row1;
        ProfScope ps(m, 0, st);
        hv_paper_kernel<T, false, 1><<<dim3((unsigned)bps, (unsigned)gy), kPaperThreads, (size_t)D.w_up * 4, st>>>(D, A);
    };
    if (m->dtype == HUBBARD_F32) launch(float{}); else launch(double{});
    return after_launch(m);
}

int lanczos_shard_update(hubbard_model *m, int mode, void *inout_dev, const void *other_dev, const void *f_dev, int64_t n,
                         double coef, double *result_dev, void *stream)
{
    int rc = check_device_model(m);
    if (rc) return rc;
    if (mode < 0 || mode > 2 || !inout_dev || n < 0 || !std::isfinite(coef)) return HUBBARD_ERR_INVALID;
    if ((mode == 0 && (!other_dev || !f_dev)) || (mode == 1 && !f_dev) || (mode != 2 && !result_dev)) return HUBBARD_ERR_INVALID;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int grid = lanczos_vec_grid(m, n);
    if ((rc = ensure_partials(m, grid))) return rc;
    if (!m->d_scal) CU_TRY(m, cudaMalloc((void **)&m->d_scal, sizeof(LanczosScalars)));
    if (!m->shard_ticket) {
        CU_TRY(m, cudaMalloc((void **)&m->shard_ticket, sizeof(unsigned)));
        CU_TRY(m, cudaMemsetAsync(m->shard_ticket, 0, sizeof(unsigned), st));
    }
    auto launch = [&](auto tag) {
        using T = decltype(tag);
        T *io = static_cast<T *>(inout_dev);
        const T *ot = static_cast<const T *>(other_dev), *ff = static_cast<const T *>(f_dev);
        ProfScope ps(m, 3, st);
        if (mode == 0) shard_update_kernel<T, 0><<<grid, kVecThreads, 0, st>>>(io, ot, ff, n, coef, m->d_partial, m->shard_ticket, result_dev);
        else if (mode == 1) shard_update_kernel<T, 1><<<grid, kVecThreads, 0, st>>>(io, ot, ff, n, coef, m->d_partial, m->shard_ticket, result_dev);
        else shard_update_kernel<T, 2><<<grid, kVecThreads, 0, st>>>(io, ot, ff, n, coef, m->d_partial, m->shard_ticket, result_dev);
    };
    if (m->dtype == HUBBARD_F32) launch(float{}); else launch(double{});
    return after_launch(m);
}

int lanczos_shard_update_noalloc(hubbard_model *m, int mode, void *inout_dev, const void *other_dev, const void *f_dev,
                                 int64_t n, double coef, double *result_dev, void *stream)
{
    int rc = check_device_model(m);
    if (rc) return rc;
    if (mode < 0 || mode > 2 || !inout_dev || n < 0 || !std::isfinite(coef)) return HUBBARD_ERR_INVALID;
    if ((mode == 0 && (!other_dev || !f_dev)) || (mode == 1 && !f_dev) || (mode != 2 && !result_dev)) return HUBBARD_ERR_INVALID;
    if (n > HUBBARD_NOALLOC_MAX_N) return HUBBARD_ERR_TOO_LARGE;     // more blocks than the fixed array has partials
    if (!m->noalloc_scratch) return HUBBARD_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int grid = (int)std::max<int64_t>(1, (n + HUBBARD_NOALLOC_CHUNK - 1) / HUBBARD_NOALLOC_CHUNK);   // <= MAX_BLOCKS
    // the array keeps whatever the last call (of any model on this GPU) left: the counter must start at zero; the
    // partials need not (every block writes its own before it takes a ticket)
    unsigned *ticket = static_cast<unsigned *>(m->noalloc_scratch);
    double *partials = reinterpret_cast<double *>(static_cast<unsigned char *>(m->noalloc_scratch) + 256);
    if (mode != 2) CU_TRY(m, cudaMemsetAsync(ticket, 0, 256, st));
    auto launch = [&](auto tag) {
        using T = decltype(tag);
        T *io = static_cast<T *>(inout_dev);
        const T *ot = static_cast<const T *>(other_dev), *ff = static_cast<const T *>(f_dev);
        if (mode == 0) shard_update_kernel<T, 0><<<grid, kVecThreads, 0, st>>>(io, ot, ff, n, coef, partials, ticket, result_dev);
        else if (mode == 1) shard_update_kernel<T, 1><<<grid, kVecThreads, 0, st>>>(io, ot, ff, n, coef, partials, ticket, result_dev);
        else shard_update_kernel<T, 2><<<grid, kVecThreads, 0, st>>>(io, ot, ff, n, coef, partials, ticket, result_dev);
    };
    if (m->dtype == HUBBARD_F32) launch(float{}); else launch(double{});
    return after_launch(m);
}

int hubbard_apply_host(hubbard_model *m, const void *x_host, void *y_host, void *stream)
{
    int rc = check_device_model(m);
    if (rc) return rc;
    if (!x_host || !y_host) return HUBBARD_ERR_INVALID;
    if ((rc = ensure_stage(m, 0)) || (rc = ensure_stage(m, 1))) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t bytes = (size_t)model_dim(m) * elem_size(m);
    CU_TRY(m, cudaMemcpyAsync(m->stage[0], x_host, bytes, cudaMemcpyHostToDevice, st));
    if ((rc = hubbard_apply(m, m->stage[0], m->stage[1], stream))) return rc;
    CU_TRY(m, cudaMemcpyAsync(y_host, m->stage[1], bytes, cudaMemcpyDeviceToHost, st));
    CU_TRY(m, cudaStreamSynchronize(st));
    return HUBBARD_OK;
}

int lanczos_run_host(hubbard_model *m, const void *v0_host, int iters, double *alpha_host, double *beta_host,
                     int *iters_done, void *stream)
{
    int rc = check_device_model(m);
    if (rc) return rc;
    if (!v0_host) return HUBBARD_ERR_INVALID;
    if ((rc = ensure_stage(m, 0))) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    CU_TRY(m, cudaMemcpyAsync(m->stage[0], v0_host, (size_t)model_dim(m) * elem_size(m), cudaMemcpyHostToDevice, st));
    return lanczos_run(m, m->stage[0], iters, alpha_host, beta_host, iters_done, stream);
}

int hubbard_get_basis(const hubbard_model *m, int spin, uint32_t *states_host)
{
    if (!m || !states_host || (spin != 0 && spin != 1)) return HUBBARD_ERR_INVALID;
    const SpinTable &tab = spin == 0 ? m->up : m->dn;
    std::memcpy(states_host, tab.states.data(), tab.states.size() * sizeof(uint32_t));
    return HUBBARD_OK;
}

int hubbard_get_hops(const hubbard_model *m, int spin, int *width, int32_t *cols_host, double *vals_host)
{
    if (!m || (spin != 0 && spin != 1) || (!width && !cols_host)) return HUBBARD_ERR_INVALID;
    if ((cols_host == nullptr) != (vals_host == nullptr)) return HUBBARD_ERR_INVALID;
    try {
        canonical_ell(spin == 0 ? m->up : m->dn, m->t, width, cols_host, vals_host);
    } catch (const std::bad_alloc &) {
        return HUBBARD_ERR_HOST_OOM;
    }
    return HUBBARD_OK;
}

int hubbard_get_gather_table(const hubbard_model *m, int spin, int lanes, int R, int sorted, int *slots, int64_t *ld,
                             uint32_t *entries_host, int32_t *counts_host, uint16_t *warp_slots_host, int32_t *perm_host,
                             int64_t *conflicts, int64_t *wavefronts)
{
    if (!m || (spin != 0 && spin != 1) || lanes < 0 || lanes > 32 || (lanes & (lanes - 1)) != 0) return HUBBARD_ERR_INVALID;
    if (R != 1 && R != 2 && R != 4) return HUBBARD_ERR_INVALID;
    const SpinTable &tab = spin == 0 ? m->up : m->dn;
    try {
        GatherTable T;
        build_gather_table(tab, lanes, R, sorted != 0, T, sorted == 2 ? m->bonds.data() : nullptr,
                           sorted == 2 ? (int)(m->bonds.size() / 2) : 0);
        if (slots) *slots = T.w;
        if (ld) *ld = T.ld;
        if (conflicts) *conflicts = T.conflicts;
        if (wavefronts) *wavefronts = T.wavefronts;
        if (entries_host) std::memcpy(entries_host, T.ent.data(), T.ent.size() * sizeof(uint32_t));
        if (counts_host) std::memcpy(counts_host, T.cnt.data(), T.cnt.size() * sizeof(int32_t));
        if (warp_slots_host) std::memcpy(warp_slots_host, T.wslots.data(), T.wslots.size() * sizeof(uint16_t));
        if (perm_host) std::memcpy(perm_host, T.perm.data(), T.perm.size() * sizeof(int32_t));
    } catch (const std::bad_alloc &) {
        return HUBBARD_ERR_HOST_OOM;
    }
    return HUBBARD_OK;
}

// ---- development / test knobs (DebugOptions, model.h)
namespace {
struct OptKey { const char *name; int hub::DebugOptions::*field; bool layout; int lo, hi; };
const OptKey kOptKeys[] = {
    {"gather_R", &hub::DebugOptions::gather_R, true, 0, 4},
    {"gather_nosched", &hub::DebugOptions::gather_nosched, true, 0, 1},
    {"gather_nosort", &hub::DebugOptions::gather_nosort, true, 0, 1},
    {"gather_nosymmetry", &hub::DebugOptions::gather_nosymmetry, true, 0, 1},
    {"gather_ctas", &hub::DebugOptions::gather_ctas, false, 1, 4},
    {"gather_fold", &hub::DebugOptions::gather_fold, false, 0, 2},
    {"gather_tmem_entries", &hub::DebugOptions::gather_tmem_entries, false, 0, 1},
    {"apply_pure_gather", &hub::DebugOptions::apply_pure_gather, false, 0, 1},
    {"twosweep_old_row", &hub::DebugOptions::twosweep_old_row, false, 0, 1},
    {"row_R", &hub::DebugOptions::row_R, false, 0, 4},
    {"strip_mb", &hub::DebugOptions::strip_mb, false, 1, 1024},
    {"strip_rb", &hub::DebugOptions::strip_rb, false, 0, 1 << 20},
    {"persist_max_dim", &hub::DebugOptions::persist_max_dim, false, 0, 1 << 30},
    {"force_cluster_row", &hub::DebugOptions::force_cluster_row, true, 0, 1},
    {"no_cluster_row", &hub::DebugOptions::no_cluster_row, true, 0, 1},
    {"cluster_R", &hub::DebugOptions::cluster_R, true, 0, 4},
    {"cluster_NC", &hub::DebugOptions::cluster_NC, true, 0, 4},
    {"paper_subvectors", &hub::DebugOptions::paper_subvectors, false, 1, 4},
};
}  // namespace

int hubbard_debug_set(hubbard_model *m, const char *key, int value)
{
    if (!m || !key) return HUBBARD_ERR_INVALID;
    for (const OptKey &k : kOptKeys) {
        if (std::strcmp(key, k.name) != 0) continue;
        if (value < k.lo || value > k.hi) return HUBBARD_ERR_INVALID;
        if (m->opt.*(k.field) == value) return HUBBARD_OK;
        m->opt.*(k.field) = value;
        if (k.layout && m->has_device) {
            const int rc = upload_layout_tables(m);
            if (rc) return rc;
            if (m->variant == HUBBARD_VARIANT_GATHER && !gather_fits(m)) m->variant = HUBBARD_VARIANT_AUTO;
        }
        return HUBBARD_OK;
    }
    return HUBBARD_ERR_INVALID;
}

int hubbard_debug_get(const hubbard_model *m, const char *key, int *value)
{
    if (!m || !key || !value) return HUBBARD_ERR_INVALID;
    for (const OptKey &k : kOptKeys)
        if (std::strcmp(key, k.name) == 0) { *value = m->opt.*(k.field); return HUBBARD_OK; }
    // what the library resolved (read-only)
    if (!std::strcmp(key, "resolved_variant")) { *value = m->has_device ? resolve_variant(m) : m->variant; return HUBBARD_OK; }
    if (!std::strcmp(key, "resolved_gather_R")) { *value = m->gather_R; return HUBBARD_OK; }
    if (!std::strcmp(key, "resolved_gather_fold")) { *value = m->has_device ? gather_fold_cols(m) : 0; return HUBBARD_OK; }
    if (!std::strcmp(key, "resolved_gather_symmetry")) { *value = m->gather_symmetry; return HUBBARD_OK; }
    if (!std::strcmp(key, "resolved_cluster_row")) { *value = m->cluster_row; return HUBBARD_OK; }
    if (!std::strcmp(key, "resolved_cluster_R")) { *value = m->cluster_R; return HUBBARD_OK; }
    if (!std::strcmp(key, "resolved_cluster_NC")) { *value = m->cluster_NC; return HUBBARD_OK; }
    return HUBBARD_ERR_INVALID;
}

int hubbard_profile(hubbard_model *m, int enable)
{
    if (!m) return HUBBARD_ERR_INVALID;
    for (auto &r : m->prof) { m->event_pool.push_back(r.e0); m->event_pool.push_back(r.e1); }
    m->prof.clear();
    for (int k = 0; k < HUBBARD_N_KCLASS; ++k) { m->prof_launches[k] = 0; m->prof_ms[k] = 0.0; }
    m->profiling = enable != 0;
    return HUBBARD_OK;
}

int hubbard_kernel_times(hubbard_model *m, int64_t *launches, double *ms)
{
    if (!m || !launches || !ms) return HUBBARD_ERR_INVALID;
    for (auto &r : m->prof) {
        CU_TRY(m, cudaEventSynchronize(r.e1));
        float t = 0.f;
        CU_TRY(m, cudaEventElapsedTime(&t, r.e0, r.e1));
        m->prof_launches[r.kclass] += 1;
        m->prof_ms[r.kclass] += (double)t;
        m->event_pool.push_back(r.e0);
        m->event_pool.push_back(r.e1);
    }
    m->prof.clear();
    for (int k = 0; k < HUBBARD_N_KCLASS; ++k) { launches[k] = m->prof_launches[k]; ms[k] = m->prof_ms[k]; }
    return HUBBARD_OK;
}

int64_t hubbard_launch_count(const hubbard_model *m) { return m ? m->launches : 0; }
int hubbard_last_cuda_error(const hubbard_model *m) { return m ? m->last_cuda_error : 0; }

const char *hubbard_strerror(int code)
{
    switch (code) {
        case HUBBARD_OK: return "ok";
        case HUBBARD_ERR_INVALID: return "invalid argument";
        case HUBBARD_ERR_HOST_OOM: return "out of host memory";
        case HUBBARD_ERR_DEVICE_OOM: return "out of device memory";
        case HUBBARD_ERR_CUDA: return "CUDA error (see hubbard_last_cuda_error)";
        case HUBBARD_ERR_NO_DEVICE: return "model has no device state (hubbard_create_host)";
        case HUBBARD_ERR_UNSUPPORTED: return "sector too large for the index types used";
        case HUBBARD_ERR_TOO_LARGE:
            return "n exceeds HUBBARD_NOALLOC_MAX_N = 268435456 elements: the no-alloc entry point's scratch is a fixed array";
        default: return "unknown error";
    }
}

}  // extern "C"
