/*
 * hubbard.h — C ABI of libhubbard_b200: the hot path of Siro & Harju,
 * "Exact diagonalization of the Hubbard model on graphics processing units"
 * (arxiv 1204.3425) for NVIDIA B200 (sm_100a).
 *
 * What the library computes
 *   H = -t sum_<ij>,s (c+_is c_js + h.c.) + U sum_i n_iup n_idn       PAPER.md:23 (eq. 1-2)
 *   in the fixed (N_up, N_dn) sector, basis ordered as in
 *   PAPER.md:41-71 (eq. 4-8): up operators left of down operators, sites
 *   ascending, state index J = i_up * dim_dn + i_dn with i_s the position of the
 *   spin's bit pattern in the ascending list of N_s-bit numbers with N_s bits set.
 *   The state vector is therefore a row-major dim_up x dim_dn matrix V
 *   (Fig. 2) and
 *       H v = (H_up (x) I) v + (I (x) H_dn) v + U popcount(up & dn) o v
 *   (eq. 14; Algorithms 2-4), fused with the
 *   Lanczos updates of Algorithm 1 in its two-vector form
 *   (eq. 12-13).
 *
 * Conventions
 *   - All functions return 0 (HUBBARD_OK) or a negative error code; nothing
 *     throws, aborts or keeps global state.  hubbard_strerror() names a code.
 *   - "host" pointers are ordinary CPU memory, "device" pointers are CUDA
 *     device memory of the current device; the caller owns every buffer it
 *     passes in.  The model owns its tables and its Lanczos work vectors.
 *   - dtype: HUBBARD_F32 (0) or HUBBARD_F64 (1) is the storage AND arithmetic
 *     type of state vectors; alpha/beta and all reductions are double.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default
 *     stream).
 *   - There is no CPU fallback: every compute call needs a CUDA device and
 *     fails with HUBBARD_ERR_CUDA / HUBBARD_ERR_NO_DEVICE otherwise.
 */
#ifndef HUBBARD_B200_H
#define HUBBARD_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hubbard_model hubbard_model;

enum {
    HUBBARD_F32 = 0,
    HUBBARD_F64 = 1
};

enum {
    HUBBARD_OK = 0,
    HUBBARD_ERR_INVALID = -1,    /* bad argument (range, null pointer, aliasing) */
    HUBBARD_ERR_HOST_OOM = -2,   /* host allocation failed */
    HUBBARD_ERR_DEVICE_OOM = -3, /* cudaMalloc failed */
    HUBBARD_ERR_CUDA = -4,       /* any other CUDA error; see hubbard_last_cuda_error */
    HUBBARD_ERR_NO_DEVICE = -5,  /* model was made by hubbard_create_host: no device state */
    HUBBARD_ERR_UNSUPPORTED = -6, /* sector too large for the index types used */
    HUBBARD_ERR_TOO_LARGE = -7   /* lanczos_shard_update_noalloc: n > HUBBARD_NOALLOC_MAX_N (its scratch is a fixed array) */
};

/* Kernel variants selectable with hubbard_set_variant (for measurement; every
 * variant computes the same H v). */
enum {
    HUBBARD_VARIANT_AUTO = 0,    /* library picks per model (default) */
    HUBBARD_VARIANT_PAPER = 1,   /* Algorithms 2-4 restated: one thread per element, one fused kernel (or four
                                    sub-vectors per block: hubbard_debug_set "paper_subvectors") */
    HUBBARD_VARIANT_TWOSWEEP = 2,/* row sweep (down term + diagonal, row staged in shared memory)
                                    + strip sweep (up term over L2-resident column strips) */
    HUBBARD_VARIANT_GATHER = 3,  /* symmetric gather sweeps: R whole rows (down term) then R whole
                                    columns (up term) staged interleaved in shared memory; in
                                    lanczos_run the vector updates are folded into the two sweeps
                                    (five work vectors in tile-major layouts).  INVALID if a row or column of V
                                    does not fit in shared memory. */
    HUBBARD_VARIANT_PERSIST = 4  /* small sectors: the whole Lanczos loop in ONE cooperative kernel, the two
                                    reductions of an iteration as grid-wide barriers (plain hubbard_apply uses
                                    the PAPER kernel).  AUTO picks it for dim <= 2^17. */
};

/* ---- construction ("first, we prepare the data on the host") ----
 *
 * hubbard_create: enumerate both spin sectors, build the
 * per-spin hopping tables with fermionic signs (eq. 9-10;
 * element = -t * (-1)^(same-spin electrons on sites strictly between the two
 * ends of the bond)), upload them, and return a model in *out.
 *   n_sites  1..32       number of lattice sites N_s (site k = bit k)
 *   n_up,n_dn 0..n_sites electrons per spin
 *   bonds    host array of 2*n_bonds site ids: undirected neighbour pairs, each
 *            listed once; both hop directions are generated ("+ h.c.").  A pair
 *            listed twice adds (effective 2t).  i == j is invalid.
 *   t, U     couplings of eq. (2)
 *   dtype    HUBBARD_F32 / HUBBARD_F64
 * Errors: INVALID (ranges, null), UNSUPPORTED (dim_up or dim_dn >= 2^31 - 1),
 * HOST_OOM, DEVICE_OOM, CUDA.  On error *out is NULL.
 *
 * hubbard_create_host: the host half only (basis + tables, no CUDA call) for
 * inspection with hubbard_get_basis / hubbard_get_hops on a machine without a
 * GPU; compute calls on such a model return HUBBARD_ERR_NO_DEVICE.
 */
int hubbard_create(hubbard_model **out, int n_sites, int n_up, int n_dn,
                   const int32_t *bonds, int n_bonds, double t, double U, int dtype);
int hubbard_create_host(hubbard_model **out, int n_sites, int n_up, int n_dn,
                        const int32_t *bonds, int n_bonds, double t, double U, int dtype);

/* Frees tables, work vectors and the model itself.  NULL is allowed. */
void hubbard_destroy(hubbard_model *m);

/* dim_up = C(N_s,N_up), dim_dn = C(N_s,N_dn) (eq. 5);
 * dim = dim_up*dim_dn may exceed 2^31.  Either output pointer may be NULL. */
int hubbard_dims(const hubbard_model *m, int64_t *dim_up, int64_t *dim_dn);

/* Change U without rebuilding tables (the diagonal is never stored,
 * PAPER.md:198,303-317). */
int hubbard_set_U(hubbard_model *m, double U);

/* Select the kernel variant (HUBBARD_VARIANT_*). */
int hubbard_set_variant(hubbard_model *m, int variant);

/* ---- the hot path ----
 *
 * hubbard_apply: y = H x.  x_dev, y_dev: device arrays of
 * dim elements of the model's dtype, element J = i_up*dim_dn + i_dn (eq. 7),
 * 16-byte aligned, not aliased (INVALID if x_dev == y_dev).  Enqueued on
 * `stream`; returns without synchronising.
 */
int hubbard_apply(hubbard_model *m, const void *x_dev, void *y_dev, void *stream);

/* lanczos_run: Algorithm 1 with the two-vector update of
 * eq. 13, H f_j fused with "- b_j f_{j-1}" and the a_j dot
 * product, "q - a_j f_j" fused with the b_{j+1} norm; normalisation is carried
 * as a scalar into the next iteration.
 *   v0_dev      device, dim elements of the model's dtype: start vector f_1; need
 *               not be normalised; not modified.
 *   iters       number of iterations m requested (>= 0)
 *   alpha_host  host, iters doubles: alpha_host[j] = a_{j+1}
 *   beta_host   host, iters doubles: beta_host[j]  = b_{j+2}
 *               (T_m of PAPER.md:150 = diag alpha[0..m-1], off-diag beta[0..m-2])
 *   iters_done  host, may be NULL: iterations completed; < iters on breakdown
 *               (Algorithm 1 lines 8-10, read as b_{j+1} <= tau*max(1,max_k|a_k|)
 *               or not finite, tau = 1e-10 for f64 / 1e-5 for f32; see
 *               lanczos_set_tau).
 * Work vectors (2 * dim elements; 5 * dim for variant GATHER) are allocated on
 * first use and kept.
 * The call enqueues everything on `stream`, then synchronises it and fills the
 * host arrays.  Errors: INVALID, DEVICE_OOM, CUDA, NO_DEVICE.
 */
int lanczos_run(hubbard_model *m, const void *v0_dev, int iters,
                double *alpha_host, double *beta_host, int *iters_done, void *stream);

/* lanczos_run_until: lanczos_run with the convergence check of PAPER.md:146
 * ("the convergence of the ground state energy can be checked after each
 * iteration").  Every `check_every` iterations (>= 1) the coefficients so far
 * are brought to the host, E_0^(m) = lambda_min(T_m) is computed and the run
 * stops when |E_0^(m) - E_0^(m - check_every)| <= tol * max(1, |E_0^(m)|), on
 * breakdown, or after max_iters iterations.  alpha_host / beta_host (max_iters
 * doubles each) and iters_done are as in lanczos_run; *e0 (may be NULL) =
 * lambda_min(T_m) for m = iters_done.  Each check synchronises the stream. */
int lanczos_run_until(hubbard_model *m, const void *v0_dev, int max_iters, int check_every, double tol,
                      double *alpha_host, double *beta_host, int *iters_done, double *e0, void *stream);

/* lanczos_ground_state: the approximate ground-state VECTOR after `iters`
 * Lanczos iterations.  The two-vector scheme discards the Lanczos basis
 * (PAPER.md:154), so the run is done twice: pass 1 gives T_m, the host computes
 * its lowest eigenvector y, pass 2 repeats the identical run
 * (all reductions are deterministic) and accumulates psi = sum_j y_j f_j.
 *   psi_dev  device, dim elements of the model's dtype, row-major (element
 *            J = i_up*dim_dn + i_dn), caller-owned, 16-byte aligned, != v0_dev;
 *            normalised to |psi| = 1 on return.
 *   e0       may be NULL: lambda_min(T_m), m = *iters_done (< iters on breakdown)
 * Synchronises the stream before returning. */
int lanczos_ground_state(hubbard_model *m, const void *v0_dev, int iters, void *psi_dev, double *e0, int *iters_done,
                         void *stream);

/* lanczos_propagate: Krylov (Lanczos) propagation with the same H v ("time propagation"):
 *   out = exp(-(tau + i t) H) v0  ~  |v0| V_m exp(-(tau + i t) T_m) e_1,   m = iters (fewer on breakdown)
 * for a REAL start vector v0 (tau: imaginary time, t: real time).  out_re_dev / out_im_dev: device, dim elements
 * of the model's dtype, row-major, caller-owned, distinct from v0 and from each other; out_im_dev may be NULL
 * (e.g. t == 0).  Pass 1 is lanczos_run, the host exponentiates T_m (full tridiagonal eigen-decomposition), each
 * output part is one more identical run accumulating sum_j y_j f_j.  Synchronises the stream.
 * (v0 must differ from the outputs here; lanczos_propagate_complex allows in-place continuation.) */
int lanczos_propagate(hubbard_model *m, const void *v0_dev, int iters, double tau, double t, void *out_re_dev,
                      void *out_im_dev, int *iters_done, void *stream);

/* lanczos_propagate_complex: the same for a COMPLEX start vector psi = re_in + i im_in (im_in_dev may be NULL = 0), so
 * that a propagation can be continued: out = exp(-(tau + i t) H) psi.  The output buffers may be the input buffers
 * (in-place continuation), but out_re_dev != out_im_dev; both outputs are required.  H is real symmetric, so this is
 * REAL Lanczos on the stacked vector [re ; im] with diag(H, H) and the real inner product - the library runs it as
 * the same lattice with the up sector listed twice through the unchanged kernels (a second model of twice the size
 * and three buffers of 2 * dim elements are allocated on first use and kept).  *iters_done as above.  Synchronises. */
int lanczos_propagate_complex(hubbard_model *m, const void *re_in_dev, const void *im_in_dev, int iters, double tau, double t,
                              void *out_re_dev, void *out_im_dev, int *iters_done, void *stream);

/* ---- row-sharded H v and Lanczos pieces (several GPUs, one model per rank; "multi-GPU ... feasible") ----
 * V is split by rows (up index): rank r owns rows [row0, row1).  The down term, the diagonal and the vector updates are
 * local to the rows; the up term reads rows of every rank, so one H v needs the FULL x (the caller all-gathers the
 * shards - the exchange step - and all-reduces the two scalars of an iteration).
 *
 * hubbard_apply_rows: y_rows = rows [row0, row1) of H x.  x_full_dev: all dim elements; y_rows_dev: (row1 - row0) *
 * dim_dn elements, row a at (a - row0) * dim_dn; 16-byte aligned, not aliased.  Algorithms 2-4 per element (the
 * kernel of variant PAPER restricted to the rows).  Enqueued on `stream`.
 *
 * lanczos_shard_update: one vector update of Algorithm 1 on a shard of n elements of the model's dtype, the scalar
 * given by the caller, the shard's partial sum left in *result_dev (a device double, fixed summation order):
 *   mode 0   inout = other - coef * inout   (line 4 with eq. 13: q = H f_j - b_j f_{j-1} over f_{j-1}),  *result = inout . f
 *   mode 1   inout = inout - coef * f       (line 6),                                                    *result = |inout|^2
 *   mode 2   inout = coef * inout           (line 11; other, f, result unused)
 * Enqueued on `stream`; nothing is synchronised. */
int hubbard_apply_rows(hubbard_model *m, const void *x_full_dev, void *y_rows_dev, int64_t row0, int64_t row1, void *stream);
int lanczos_shard_update(hubbard_model *m, int mode, void *inout_dev, const void *other_dev, const void *f_dev, int64_t n,
                         double coef, double *result_dev, void *stream);

/* lanczos_shard_update_noalloc: lanczos_shard_update for callers that must not allocate (CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc).  Same arguments, same arithmetic per element (Algorithm 1 lines
 * 4-7 and 11, eq. 13), same fixed-order fp64 reduction - but the per-block partial sums and the
 * arrival counter live in ONE fixed array inside the library (static __device__, HUBBARD_NOALLOC_SCRATCH_BYTES = 256 +
 * 8 * 8192 bytes, held by every GPU that loads the library until the process exits) instead of buffers the model
 * allocates on first use.  The call makes no cudaMalloc / cudaFree, creates no event or stream and synchronises
 * nothing: it enqueues one 256-byte memset (the counter must start at zero) and one kernel on `stream`.  The array's
 * device address is resolved once per device when a model is created on it (hubbard_create).
 *   - one block per HUBBARD_NOALLOC_CHUNK = 32768 elements, one partial per block, hence
 *     n <= HUBBARD_NOALLOC_MAX_N = 8192 * 32768 = 268 435 456 elements; a larger n returns HUBBARD_ERR_TOO_LARGE and
 *     nothing is enqueued (all three modes).  The partial sums are cut differently from lanczos_shard_update's, so
 *     *result_dev agrees with it to rounding (fp64 accumulation in both), the updated vector bit for bit.
 *   - the array is shared by EVERY call on that GPU, of every model, and keeps the last call's contents: two calls
 *     that may overlap on the GPU (different streams, no dependency between them) RACE on it.  Serialise them.
 *   - hubbard_profile does not see these launches (timing them would create events). */
#define HUBBARD_NOALLOC_CHUNK 32768
#define HUBBARD_NOALLOC_MAX_BLOCKS 8192
#define HUBBARD_NOALLOC_MAX_N ((int64_t)HUBBARD_NOALLOC_MAX_BLOCKS * HUBBARD_NOALLOC_CHUNK)
#define HUBBARD_NOALLOC_SCRATCH_BYTES (256 + 8 * HUBBARD_NOALLOC_MAX_BLOCKS)
int lanczos_shard_update_noalloc(hubbard_model *m, int mode, void *inout_dev, const void *other_dev, const void *f_dev,
                                 int64_t n, double coef, double *result_dev, void *stream);

/* Breakdown threshold tau (>= 0; 0 = the paper's literal "b = 0" test). */
int lanczos_set_tau(hubbard_model *m, double tau);

/* ---- same calls with HOST vectors (copies inside): the end-to-end entry ----
 * x_host/y_host/v0_host: host arrays of dim elements of the model's dtype.
 * The library stages them through its own device buffers (allocated on first
 * use, kept), runs the device path above on `stream`, copies the result back
 * and synchronises. */
int hubbard_apply_host(hubbard_model *m, const void *x_host, void *y_host, void *stream);
int lanczos_run_host(hubbard_model *m, const void *v0_host, int iters,
                     double *alpha_host, double *beta_host, int *iters_done, void *stream);

/* ---- introspection for bit-exact table parity ----
 *
 * hubbard_get_basis: states_host[i] = i-th bit pattern of spin `spin`
 * (0 = up, 1 = down), dim_spin entries, ascending.
 *
 * hubbard_get_hops: the per-spin hopping matrix H_spin of eq. 14 in canonical
 * ELL form, independent of the device layout: row-major dim_spin x width,
 * entries of a row sorted by ascending column, duplicates merged, exact zeros
 * dropped, padding col = -1 / val = 0 (PAPER.md:208-230 describes ELL; the
 * paper pads with 0).  Call with cols_host == NULL to obtain only *width
 * (= max nonzeros per row).
 */
int hubbard_get_basis(const hubbard_model *m, int spin, uint32_t *states_host);
int hubbard_get_hops(const hubbard_model *m, int spin, int *width,
                     int32_t *cols_host, double *vals_host);

/* hubbard_get_gather_table: the DEVICE layout of one spin's hop table as variant
 * GATHER uses it (host computation only; works on hubbard_create_host models):
 * the ELL format of PAPER.md:208-230 over an INTERNAL order of the spin's basis
 * states (position p holds state perm[p] of the ascending list of PAPER.md:63-67;
 * sorted == 2: orbits of a group of `lanes` lattice symmetries as aligned groups,
 * ordered by descending hop count - equal row lengths inside a group and no bank
 * conflicts by construction, see csrc/gather_tables.h - falling back to sorted ==
 * 1 when the bond list has no such group; sorted == 1: aligned groups of `lanes`
 * consecutive states ordered by descending hop count; sorted == 0: perm =
 * identity, what the row-major vectors of hubbard_apply need), with
 * batches of 8 entries of one position contiguous - entry k of position p at
 * [((k / 8) * ld + p) * 8 + k % 8], entry = target_position * 2 + neg (element =
 * t * (neg ? -1 : +1)) - and a position's entries placed in its
 * slots so that the `lanes` lanes served by one shared-memory wavefront (8, 16 or
 * 32; 0 = keep bond order) hit distinct banks.  R (1, 2 or 4) is the tile height:
 * the tile holds n_pos = dim_spin rounded up to R positions followed by `lanes`
 * zero slots, and padding entries have target_position >= n_pos.
 * Call first with the array arguments NULL to obtain *slots (entries per position
 * in the table, a multiple of 8) and *ld (a multiple of 32, >= n_pos); then pass
 *   entries_host[*ld * *slots], counts_host[*ld] (last slot holding a real entry + 1),
 *   warp_slots_host[*ld / 32] (the EXACT number of slots every lane of that warp of
 *   32 positions walks; slots below it hold real or zero-slot entries),
 *   perm_host[*ld] (position -> state index, -1 for padding positions).
 * *conflicts = entries that share a bank with another lane of their wavefront;
 * *wavefronts = shared-memory wavefronts one tile's gather costs in this layout
 * (sum over warps of warp_slots * 32 / lanes, plus the conflicts' replays). */
int hubbard_get_gather_table(const hubbard_model *m, int spin, int lanes, int R, int sorted, int *slots, int64_t *ld,
                             uint32_t *entries_host, int32_t *counts_host, uint16_t *warp_slots_host, int32_t *perm_host,
                             int64_t *conflicts, int64_t *wavefronts);

/* ---- host utility, off the hot path ----
 * e0 = smallest eigenvalue of the symmetric tridiagonal T_m with diagonal
 * alpha[0..m-1] and off-diagonal beta[0..m-2]; m >= 1. */
int lanczos_ground_energy(const double *alpha, const double *beta, int m, double *e0);
/* Same, plus the eigenvector y (m doubles, unit norm, y[0] >= 0) of that eigenvalue (inverse iteration); e0 may be NULL. */
int lanczos_ground_vector(const double *alpha, const double *beta, int m, double *e0, double *y);
/* y = exp(-(tau + i t) T_m) e_1 as real and imaginary parts (m doubles each); host, O(m^3). */
int lanczos_expm_e1(const double *alpha, const double *beta, int m, double tau, double t, double *y_re, double *y_im);

/* ---- measurement hooks ----
 * hubbard_profile(m, 1) makes every later kernel launch of this model be
 * bracketed by CUDA events on its stream; hubbard_kernel_times then returns,
 * per kernel class, the number of launches and the summed device time in ms
 * since the last hubbard_profile call (it synchronises the recorded events).
 * Classes: 0 = H v kernel(s) of variant PAPER and the cooperative kernel of PERSIST, 1 = row sweep (down term),
 * 2 = strip / column sweep (up term), 3 = Lanczos axpy+norm or closing norm
 * sweep, 4 = scalar/finalise kernels, 5 = setup (copy, initial norm).
 * Arrays have HUBBARD_N_KCLASS entries.
 * hubbard_launch_count: kernels launched by this model since creation. */
#define HUBBARD_N_KCLASS 6
int hubbard_profile(hubbard_model *m, int enable);
int hubbard_kernel_times(hubbard_model *m, int64_t *launches, double *ms);
int64_t hubbard_launch_count(const hubbard_model *m);

/* ---- development / test knobs (per model; nothing is read from the environment) ----
 * hubbard_debug_set forces one dispatch or geometry decision of this model so that a test or an A/B measurement
 * states what it forces; the defaults are what bench.py times and what production callers get.  Keys (value range):
 *   "gather_R" (0-4)          cap on the tile height R of variant GATHER, 0 = none (what a larger sector would get)
 *   "gather_nosched" (0/1)    hop entries in bond order, no bank-aware placement
 *   "gather_nosort" (0/1)     the Lanczos work vectors of variant GATHER keep the basis order
 *   "gather_nosymmetry" (0/1) their internal order comes from hop counts only (no lattice-symmetry orbits)
 *   "gather_ctas" (1-4)       CTAs per SM for small tiles
 *   "gather_fold" (0-2)       lanczos_* of variant GATHER in the folded, eight-pass form (the ROW sweep parks its tile of
 *                             u_j in tensor memory and applies "- b_{j+1} f_j" of Algorithm 1 line 4 itself): 1 (default)
 *                             where one tile fills an SM's shared memory (C4), 2 wherever the SM's 512 tensor-memory
 *                             columns suffice for its resident CTAs, 0 never = the nine-pass form (the COL sweep reads
 *                             u_j).  DESIGN.md 2 (readings) and 4.2
 *   "gather_tmem_entries" (0/1)  folded form: the COL sweep keeps the first hop-entry batch of each of its positions in
 *                             tensor memory for the whole launch (default 1; 0 = every batch is loaded from L2)
 *   "apply_pure_gather" (0/1) plain hubbard_apply as two gather sweeps instead of the hybrid
 *   "twosweep_old_row" (0/1)  AUTO's TWOSWEEP fallback keeps the first row kernel
 *   "row_R" (0-4), "strip_mb" (1-1024), "strip_rb"   geometry of variant TWOSWEEP (0 = automatic)
 *   "persist_max_dim"         largest dim that AUTO runs in the cooperative kernel
 *   "paper_subvectors" (1 or 4)  variant PAPER: sub-vectors per block = elements per thread (4 = the paper's tuned
 *                             form; any other value means 1)
 *   "force_cluster_row" (0/1), "no_cluster_row" (0/1), "cluster_R" (0-4), "cluster_NC" (0,2,4)
 *                             take / avoid the cluster row sweep of rows larger than one SM, force one (R, NC)
 * Options that change a device table layout re-upload that table (host work + cudaMemcpy; no kernel launch).
 * hubbard_debug_get returns an option, or what the library resolved for this model: "resolved_variant"
 * (HUBBARD_VARIANT_* that AUTO stands for), "resolved_gather_R", "resolved_gather_fold" (tensor-memory columns one
 * CTA of the folded ROW sweep allocates, 0 = nine-pass form), "resolved_gather_symmetry" (order of the lattice symmetry group the
 * internal order of variant GATHER was built from, 0 = none), "resolved_cluster_row", "resolved_cluster_R",
 * "resolved_cluster_NC".  Unknown key or out-of-range value: HUBBARD_ERR_INVALID. */
int hubbard_debug_set(hubbard_model *m, const char *key, int value);
int hubbard_debug_get(const hubbard_model *m, const char *key, int *value);

/* Last CUDA error code (cudaError_t as int) seen by this model, 0 if none. */
int hubbard_last_cuda_error(const hubbard_model *m);
const char *hubbard_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* HUBBARD_B200_H */
