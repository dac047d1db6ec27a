// Variant GATHER: H v as two symmetric "gather sweeps".
//
// H_hop is a Kronecker SUM (eq. 14): the down term couples
// elements of one ROW of V, the up term elements of one COLUMN.  Both sweeps
// therefore use the same device code on a tile that is closed under its term:
//
//   ROW sweep  tile = R whole rows    (a0..a0+R-1, all b)   contracts H_dn   eq. 16 + Algorithm 4
//   COL sweep  tile = R whole columns (all a, c0..c0+R-1)   contracts H_up   eq. 15
//
// The tile is staged in shared memory INTERLEAVED, Xs[i][r] (i = the contracted
// index, r = 0..R-1 the tile's rows/columns), R*sizeof(T) = 16 bytes when it
// fits, so that ONE 128-bit shared-memory load fetches the hop source of all R
// outputs a thread owns; the hop entry (Algorithms 2/3: Aj, Ax of the ELL
// format, stored so that a warp reads them coalesced: batches
// of 8 entries of one state are contiguous, batch kb of state i at
// [(kb * ld + i) * 8]) is read once per R outputs.  Padding entries point at a
// zero slot.  Every lane of a warp walks the same, EXACT number of slots (the
// table's per-warp count, gather_tables.h), so the trip count is warp-uniform
// and the last, partial batch is cut with uniform branches.
//
// "State i" below is a POSITION in the table's internal order of the spin's basis
// (gather_tables.h: groups ordered by hop count so that a warp's rows have nearly
// equal length); the Lanczos work vectors live in that order for both spins, the
// caller's row-major vectors are converted at the start / end of a run.
//
// Work vectors live in HBM in two TILE-MAJOR layouts made of 16-byte PIECES (the R
// values of one contracted position of one tile = one shared-memory slot), so
// that every tile either sweep stages is ONE contiguous block that is already its
// shared-memory image (du_p, dd_p = dim_up, dim_dn rounded up to R; padding holds
// zeros):
//   RT  piece (row tile m, column b)  at m * dd_p + b     element (a, b) at ((a / R) * dd_p + b) * R + a % R
//   CT  piece (column tile c, row a)  at c * du_p + a     element (a, b) at ((b / R) * du_p + a) * R + b % R
// A sweep reads its own layout contiguously and writes what the other sweep
// will stage in the OTHER layout: the R x R block held by R adjacent lanes is
// transposed with warp shuffles and each lane stores one piece (full 32/64-byte
// sectors, asynchronous) - all strided traffic is writes (struct Layout records
// what interleaving several tiles line by line did instead).
//
// Lanczos form (Algorithm 1 with eq. 13), no separate
// axpy/norm kernel:
//   ROW sweep of iteration j+1:  w = q_j - a_j f_j  (line 6; staged, written over
//        q_j in RT and also in CT), b_{j+1}^2 = |w|^2 (line 7),
//        z = (t H_dn + D) w -> CT; the last block records a_j, b_{j+1}, applies
//        lines 8-10 and carries f_{j+1} = w / b_{j+1} (line 11) as c = 1/b_{j+1}.
//   COL sweep of iteration j+1:  q_{j+1} = c (t H_up w + z) - b_{j+1} f_j  (line 4,
//        written over f_j in RT as in eq. 13) and a_{j+1} = q_{j+1} . f_{j+1} (line 5).
#pragma once
#include "gather_tables.h"
#include "kernels_common.cuh"

namespace hub {

constexpr int kGatherMaxThreads = 1024;  // one CTA of 1024 threads per SM, or 2-4 smaller ones when their tiles fit together
constexpr int kGatherBatch = kSlotBatch; // hop entries per batch (gather_tables.h), one batch always in flight
#ifndef GS_HOIST
#define GS_HOIST 1
#endif
#ifndef GS_L2PF
#define GS_L2PF 1
#endif
#ifndef GS_TMA_STAGE
#define GS_TMA_STAGE 1    // COL sweep: stage the tile with cp.async.bulk + mbarrier instead of per-thread loads
#endif
#ifndef GS_FOLD_LATE
#define GS_FOLD_LATE 1    // folded ROW sweep: take the parked piece back after the gather (1.96 ms) instead of before it (1.98 ms)
#endif
#ifndef GS_STAGE_UNROLL
#define GS_STAGE_UNROLL 1
#endif
constexpr int kStageUnroll = GS_STAGE_UNROLL;          // 16-byte pieces in flight per thread while staging

template <typename T>
struct GatherArgs {
    SpinDev in;             // the spin whose index is contracted (dn for ROW, up for COL)
    const uint32_t *st_out; // bit patterns of the other spin (ROW: states_up, for the diagonal)
    int64_t dim_up, dim_dn; // du, dd
    int64_t du_p, dd_p;     // rounded up to R
    double t, U;
    // plain apply: y = H x, both row-major (the ABI layout); xct, zct internal CT buffers
    const T *x;
    T *y;
    // Lanczos: Qrt holds q_j -> w, Frt holds u_j (f_j = c_j u_j) -> q_{j+1}   (RT layout)
    //          Wct <- w, Zct <- z (written by ROW, read by COL), Fct = u_j      (CT layout)
    T *Qrt, *Frt, *Wct, *Zct;
    const T *Fct;
    LanczosScalars *S;
    double *partials;
    double *alpha_out, *beta_out;
    int y_rowmajor;         // ROW sweep of hubbard_apply writes y row-major (no CT buffers): hybrid with the strip sweep
    // Lanczos, folded (eight-pass) form: tensor-memory columns the ROW sweep allocates to park u_j (0: nine-pass form,
    // the COL sweep reads u_j in CT)
    int fold_cols;
    // Folded form, COL sweep: tensor-memory columns to keep the FIRST batch of hop entries of every position this CTA's
    // threads own (the same positions in every tile) for the whole launch; 0: all entry batches come from L2
    int ent_cols;
};

template <typename T, int N>
struct alignas(sizeof(T) * N) Pack {
    T v[N];
};

// Piece index of (tile, position) in a tile-major layout whose contracted dimension has n_p positions.
// S tiles can be interleaved line by line into a super-tile (S = 1: every tile is one contiguous block).  Measured
// on C4 fp64: S = 4 turns the transposed 32-byte stores into whole 128-byte lines, which HBM
// takes at 4.6 instead of 2.9 TB/s in isolation, but the tile is then READ as sectors at a 128-byte stride - four
// times the lines per load instruction, and the sweeps are bound by load latency: 5.0 ms per iteration against 3.6
// (S = 2: 4.0 ms).  S = 1 it is.
template <typename T, int R>
struct Layout {
    static constexpr int S = 1;
    static __host__ __device__ __forceinline__ int64_t piece(int64_t tile, int64_t pos, int64_t n_p)
    {
        if constexpr (S == 1) return tile * n_p + pos;       // (R divides n_p: the general form below reduces to this)
        return (((tile / S) * (n_p / R) + pos / R) * S + tile % S) * R + pos % R;
    }
};

template <typename T> __device__ __forceinline__ T sign_one(uint32_t e);
// +1 or -1 from the low bit of an entry (1 -> -1)
template <> __device__ __forceinline__ float sign_one<float>(uint32_t e)
{
    return __uint_as_float(0x3f800000u | (e << 31));
}
template <> __device__ __forceinline__ double sign_one<double>(uint32_t e)
{
    return __hiloint2double((int)(0x3ff00000u | (e << 31)), 0);
}

// One batch of kGatherBatch hop entries of one state: contiguous bytes, read
// through the read-only path with the widest loads.
// (16-bit entries travel as the four 32-bit words they are packed in - a struct of eight uint16 makes the compiler
// re-pack them with PRMT at every copy.)
template <typename E> struct BatchOf { using type = Pack<E, kGatherBatch>; };
template <> struct BatchOf<uint16_t> { using type = Pack<uint32_t, kGatherBatch / 2>; };
template <typename E, int N>
__device__ __forceinline__ Pack<E, N> load_batch(const Pack<E, N> *p)
{
    constexpr int kBytes = (int)sizeof(E) * N;
    Pack<E, N> o;
    if constexpr (kBytes % 16 == 0) {
        uint4 u[kBytes / 16];
#pragma unroll
        for (int k = 0; k < kBytes / 16; ++k) u[k] = __ldg(reinterpret_cast<const uint4 *>(p) + k);
        memcpy(&o, u, kBytes);
    } else {
        static_assert(kBytes == 8, "batch must be 8 bytes or a multiple of 16");
        const uint2 u = __ldg(reinterpret_cast<const uint2 *>(p));
        memcpy(&o, &u, kBytes);
    }
    return o;
}

template <typename E> __device__ __forceinline__ const E *ent_ptr(const SpinDev &s);
template <> __device__ __forceinline__ const uint16_t *ent_ptr<uint16_t>(const SpinDev &s) { return s.e16; }
template <> __device__ __forceinline__ const uint32_t *ent_ptr<uint32_t>(const SpinDev &s) { return s.e32; }

// Record a_j, b_{j+1} and rotate the scalars (Algorithm 1 lines 7-11); called
// by thread 0 of the last block of a norm-producing sweep.
__device__ __forceinline__ void lanczos_rotate(LanczosScalars *S, double b2, double *alpha_out, double *beta_out)
{
    const double beta = sqrt(b2);
    bool stop = false;
    if (S->started > 0) {
        const int j = S->j;
        const double alpha = S->alpha;
        alpha_out[j] = alpha;
        beta_out[j] = beta;
        const double amax = fmax(S->amax, fabs(alpha));
        S->amax = amax;
        S->j = j + 1;
        stop = !isfinite(beta) || !(beta > S->tau * fmax(1.0, amax));      // lines 8-10, reading Q11
    } else {
        stop = !isfinite(beta) || !(beta > 0.0);                            // unusable start vector
    }
    if (stop) {
        S->stop = 1;
    } else {
        S->c_prev = S->c_cur;
        S->c_cur = 1.0 / beta;                                              // line 11, carried lazily
        S->beta = beta;
    }
    S->started += 1;
    S->ticket = 0;
}

// ------------------------------------------------------------------ bulk (TMA) staging of a contiguous tile
// cp.async.bulk moves a contiguous block global -> shared memory without occupying threads, registers or the
// LSU; completion is counted in bytes on an mbarrier in shared memory.
__device__ __forceinline__ uint32_t smem_addr_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_addr_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, unsigned bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_addr_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_addr_u32(bar))
                 : "memory");
}

// ------------------------------------------------------------------ helpers
// Streaming (evict-first, .cs) accesses for data that is used once per sweep, so that it does not displace the
// next tile's prefetched inputs in L2.  Bit masks, measured per access class on C4:
// GS_STCS 1 = w in RT, 2 = the transposed stores of the ROW sweep (-5.5 %), 4 = q of the COL sweep (-1 %);
// GS_LDCS 1 = ROW staging, 2 = COL staging (-2 %), 4 = z/u of the COL epilogue in fp32 (-3 %; +2 % in fp64: bit 8).
#ifndef GS_LDCS
#define GS_LDCS 7
#endif
#ifndef GS_STCS
#define GS_STCS 7
#endif
template <int BIT, typename P>
__device__ __forceinline__ P ld_once(const P *p)
{
    if constexpr ((GS_LDCS & BIT) == 0) {
        return *p;
    } else if constexpr (sizeof(P) == 16) {
        const float4 u = __ldcs(reinterpret_cast<const float4 *>(p));
        return *reinterpret_cast<const P *>(&u);
    } else if constexpr (sizeof(P) == 8) {
        const float2 u = __ldcs(reinterpret_cast<const float2 *>(p));
        return *reinterpret_cast<const P *>(&u);
    } else {
        const float u = __ldcs(reinterpret_cast<const float *>(p));
        return *reinterpret_cast<const P *>(&u);
    }
}
#ifndef GS_EARLY_FIRST
#define GS_EARLY_FIRST 1
#endif
// staging loads of the folded ROW sweep
#ifndef GS_PARK_UNROLL
#define GS_PARK_UNROLL 1
#endif
#ifndef GS_PARK_NA
#define GS_PARK_NA 0
#endif
template <typename P>
__device__ __forceinline__ P ld_stage(const P *p)
{
#if GS_PARK_NA
    if constexpr (sizeof(P) == 16) {
        uint32_t a, b, c, d;
        asm volatile("ld.global.L1::no_allocate.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "l"(p));
        const uint32_t u[4] = {a, b, c, d};
        P o;
        memcpy(&o, u, 16);
        return o;
    } else {
        return ld_once<1>(p);
    }
#else
    return ld_once<1>(p);
#endif
}
template <int BIT, typename P>
__device__ __forceinline__ void st_once(P *p, const P &v)
{
    if constexpr ((GS_STCS & BIT) == 0) *p = v;
    else if constexpr (sizeof(P) == 16) __stcs(reinterpret_cast<float4 *>(p), *reinterpret_cast<const float4 *>(&v));
    else if constexpr (sizeof(P) == 8) __stcs(reinterpret_cast<float2 *>(p), *reinterpret_cast<const float2 *>(&v));
    else __stcs(reinterpret_cast<float *>(p), *reinterpret_cast<const float *>(&v));
}

template <typename T, int R>
__device__ __forceinline__ T pick(const T (&v)[R], int idx)
{
    T r = v[0];
#pragma unroll
    for (int k = 1; k < R; ++k) r = (idx == k) ? v[k] : r;
    return r;
}

// R adjacent lanes (q = lane % R) hold an R x R block, lane q holding column q
// as v[r] = (row r, column q).  Returns in lane q the row q: o[c] = (row q, column c).
template <typename T, int R>
__device__ __forceinline__ Pack<T, R> block_transpose(const T (&v)[R], int q)
{
    Pack<T, R> o;
    if (R == 1) {
        o.v[0] = v[0];
        return o;
    }
    if constexpr (R == 2) {
        // lane q keeps element q of its own column and swaps the other one with its partner
        const T got = __shfl_xor_sync(0xffffffffu, q ? v[0] : v[1], 1);
        o.v[0] = q ? got : v[0];
        o.v[1] = q ? v[1] : got;
        return o;
    }
    T tmp[R];
    tmp[0] = pick<T, R>(v, q);
#pragma unroll
    for (int d = 1; d < R; ++d) tmp[d] = __shfl_xor_sync(0xffffffffu, pick<T, R>(v, q ^ d), d);
#pragma unroll
    for (int c = 0; c < R; ++c) o.v[c] = pick<T, R>(tmp, c ^ q);
    return o;
}

// Stage R rows of a ROW-MAJOR vector interleaved: each thread loads VW consecutive columns of each of the R
// rows (R vector loads in flight) and stores VW interleaved pieces.  n_in = dd must be a multiple of VW.
template <typename T, int R, int VW>
__device__ __forceinline__ void stage_rowmajor(const T *__restrict__ x, Pack<T, R> *Xs, int64_t o0, int64_t du, int64_t dd,
                                               int n_in, int n_in_p, int nthr)
{
    using PV = Pack<T, VW>;
    for (int b = (int)threadIdx.x * VW; b < n_in_p; b += nthr * VW) {
        PV in[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
#pragma unroll
            for (int c = 0; c < VW; ++c) in[r].v[c] = T(0);
            if (o0 + r < du && b < n_in) in[r] = *reinterpret_cast<const PV *>(x + (o0 + r) * dd + b);
        }
#pragma unroll
        for (int c = 0; c < VW; ++c) {
            Pack<T, R> o;
#pragma unroll
            for (int r = 0; r < R; ++r) o.v[r] = in[r].v[c];
            if (b + c < n_in_p) Xs[b + c] = o;
        }
    }
}

// acc += +-Xs[col] for one hop entry (Algorithms 2/3: sum += Ax * x[Aj])
template <typename T, int R>
__device__ __forceinline__ void hop(const unsigned char *xs_bytes, uint32_t e, T (&acc)[R])
{
    using PR = Pack<T, R>;
    const PR v = *reinterpret_cast<const PR *>(xs_bytes + (e & ~1u) * (uint32_t)(sizeof(PR) / 2));
    const T s = sign_one<T>(e);
#pragma unroll
    for (int r = 0; r < R; ++r) acc[r] = fma(s, v.v[r], acc[r]);
}

// ---- 16-bit device entries, two per 32-bit word (upload_gather_table): the EVEN entry of a word as
// position << 1 | neg in bits 0..15, the ODD one as position | neg << 15 in bits 16..31 (the matrix element is
// t * (neg ? -1 : +1)).  Chosen for what one integer instruction can do: the byte offset of either
// entry is one mask and one shift-and-add away from the word (LOP3 + LEA / LEA.HI), the sign of the odd entry is
// already where a float / the high word of a double has it, the sign of the even one is one shift-and-add (w << 31).
template <typename PR>
__device__ __forceinline__ PR lds_piece(uint32_t saddr)
{
    PR v;
    if constexpr (sizeof(PR) == 16) {
        uint32_t a, b, c, d;
        asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "r"(saddr));
        const uint32_t u[4] = {a, b, c, d};
        memcpy(&v, u, 16);
    } else if constexpr (sizeof(PR) == 8) {
        uint32_t a, b;
        asm volatile("ld.shared.v2.b32 {%0, %1}, [%2];" : "=r"(a), "=r"(b) : "r"(saddr));
        const uint32_t u[2] = {a, b};
        memcpy(&v, u, 8);
    } else {
        static_assert(sizeof(PR) == 4, "pieces are 4, 8 or 16 bytes");
        uint32_t a;
        asm volatile("ld.shared.b32 %0, [%1];" : "=r"(a) : "r"(saddr));
        memcpy(&v, &a, 4);
    }
    return v;
}
template <typename T> __device__ __forceinline__ T sign_top(uint32_t w);      // +-1 from bit 31
template <> __device__ __forceinline__ float sign_top<float>(uint32_t w) { return __uint_as_float((w & 0x80000000u) | 0x3f800000u); }
template <> __device__ __forceinline__ double sign_top<double>(uint32_t w)
{
    return __hiloint2double((int)((w & 0x80000000u) | 0x3ff00000u), 0);
}
template <typename T, int R>
__device__ __forceinline__ void hop_lo(uint32_t xs_s, uint32_t w, T (&acc)[R])      // even entry: bits 0..15
{
    using PR = Pack<T, R>;
    constexpr int SH = sizeof(PR) == 16 ? 3 : sizeof(PR) == 8 ? 2 : 1;
    const PR v = lds_piece<PR>(xs_s + ((w & 0xfffeu) << SH));
    const T s = sign_one<T>(w);                            // (w << 31): only bit 0 survives
#pragma unroll
    for (int r = 0; r < R; ++r) acc[r] = fma(s, v.v[r], acc[r]);
}
template <typename T, int R>
__device__ __forceinline__ void hop_hi(uint32_t xs_s, uint32_t w, T (&acc)[R])      // odd entry: bits 16..31
{
    using PR = Pack<T, R>;
    constexpr int SH = sizeof(PR) == 16 ? 12 : sizeof(PR) == 8 ? 13 : 14;
    const PR v = lds_piece<PR>(xs_s + ((w & 0x7fff0000u) >> SH));
    if constexpr (sizeof(T) == 8) {
        // the sign bit of the entry IS the sign bit of a double's high word: flip it into the value (one three-input
        // LOP3 per output) and add - no +-1.0 to build, exact like the multiplication by +-1
#pragma unroll
        for (int r = 0; r < R; ++r)
            acc[r] += __hiloint2double(__double2hiint(v.v[r]) ^ (int)(w & 0x80000000u), __double2loint(v.v[r]));
    } else {
        const T s = sign_top<T>(w);
#pragma unroll
        for (int r = 0; r < R; ++r) acc[r] = fma(s, v.v[r], acc[r]);
    }
}
// position and sign of entry j of a packed batch, for kernels that do not gather from a local tile
__device__ __forceinline__ uint32_t packed_pos(const Pack<uint32_t, kGatherBatch / 2> &pk, int j)
{
    const uint32_t w = pk.v[j >> 1];
    return (j & 1) ? ((w >> 16) & 0x7fffu) : ((w >> 1) & 0x7fffu);
}
template <typename T>
__device__ __forceinline__ T packed_sign(const Pack<uint32_t, kGatherBatch / 2> &pk, int j)
{
    const uint32_t w = pk.v[j >> 1];
    return (j & 1) ? sign_top<T>(w) : sign_one<T>(w);
}

// `count` (warp-uniform, 1..8) entries of a batch.
template <typename T, int R>
__device__ __forceinline__ void hop_batch_n(const unsigned char *xs_bytes, const Pack<uint32_t, kGatherBatch / 2> &pk, int count, T (&acc)[R])
{
    static_assert(kGatherBatch == 8, "a batch is four 32-bit words of two entries");
    const uint32_t xs_s = smem_addr_u32(xs_bytes);
    uint32_t w[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) w[k] = pk.v[k];
    if (count == kGatherBatch) {
#pragma unroll
        for (int k = 0; k < 4; ++k) { hop_lo<T, R>(xs_s, w[k], acc); hop_hi<T, R>(xs_s, w[k], acc); }
    } else {
        if (count & 4) {
            hop_lo<T, R>(xs_s, w[0], acc); hop_hi<T, R>(xs_s, w[0], acc);
            hop_lo<T, R>(xs_s, w[1], acc); hop_hi<T, R>(xs_s, w[1], acc);
            w[0] = w[2]; w[1] = w[3];
        }
        if (count & 2) {
            hop_lo<T, R>(xs_s, w[0], acc); hop_hi<T, R>(xs_s, w[0], acc);
            w[0] = w[1];
        }
        if (count & 1) hop_lo<T, R>(xs_s, w[0], acc);
    }
}
template <typename T, int R>
__device__ __forceinline__ void hop_batch_n(const unsigned char *xs_bytes, const Pack<uint32_t, kGatherBatch> &pk, int count, T (&acc)[R])
{
    uint32_t e[kGatherBatch];
#pragma unroll
    for (int j = 0; j < kGatherBatch; ++j) e[j] = pk.v[j];
    if (count == kGatherBatch) {
#pragma unroll
        for (int j = 0; j < kGatherBatch; ++j) hop<T, R>(xs_bytes, e[j], acc);
    } else {
        if (count & 4) {
#pragma unroll
            for (int j = 0; j < 4; ++j) { hop<T, R>(xs_bytes, e[j], acc); e[j] = e[j + 4]; }
        }
        if (count & 2) {
            hop<T, R>(xs_bytes, e[0], acc);
            hop<T, R>(xs_bytes, e[1], acc);
            e[0] = e[2];
        }
        if (count & 1) hop<T, R>(xs_bytes, e[0], acc);
    }
}

// ------------------------------------------------------------------ tensor memory as a per-thread parking buffer
// Folded Lanczos form (ROW sweep): the tile fills the shared memory, and the epilogue of a position needs the piece of
// u_j that the same thread loaded while staging it.  The SM's 256 KB of tensor memory (128 lanes x 512 columns x 4
// bytes, otherwise unused by this library) holds it: warp w owns lanes 32 (w % 4) .. + 31 (the only ones it can
// address), a thread parks its piece with tcgen05.st (SASS STTM) and takes the same piece back with tcgen05.ld
// (LDTM) - no other thread ever touches it, so no cross-thread ordering is involved.
__device__ __forceinline__ void tmem_alloc(uint32_t *slot_smem, uint32_t ncols)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_addr_u32(slot_smem)), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
template <int W> __device__ __forceinline__ void tmem_st(uint32_t taddr, const uint32_t (&v)[W]);
template <> __device__ __forceinline__ void tmem_st<1>(uint32_t taddr, const uint32_t (&v)[1])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(taddr), "r"(v[0]) : "memory");
}
template <> __device__ __forceinline__ void tmem_st<2>(uint32_t taddr, const uint32_t (&v)[2])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "r"(v[0]), "r"(v[1]) : "memory");
}
template <> __device__ __forceinline__ void tmem_st<4>(uint32_t taddr, const uint32_t (&v)[4])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3])
                 : "memory");
}
// the registers of a tcgen05.ld are valid after tcgen05.wait::ld: the wait names them so that no use moves above it
template <int W> __device__ __forceinline__ void tmem_ld(uint32_t taddr, uint32_t (&v)[W]);
template <int W> __device__ __forceinline__ void tmem_wait_ld(uint32_t (&v)[W]);
template <> __device__ __forceinline__ void tmem_ld<1>(uint32_t taddr, uint32_t (&v)[1])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v[0]) : "r"(taddr) : "memory");
}
template <> __device__ __forceinline__ void tmem_ld<2>(uint32_t taddr, uint32_t (&v)[2])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(v[0]), "=r"(v[1]) : "r"(taddr) : "memory");
}
template <> __device__ __forceinline__ void tmem_ld<4>(uint32_t taddr, uint32_t (&v)[4])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(taddr)
                 : "memory");
}
template <> __device__ __forceinline__ void tmem_wait_ld<1>(uint32_t (&v)[1])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(v[0])::"memory");
}
template <> __device__ __forceinline__ void tmem_wait_ld<2>(uint32_t (&v)[2])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(v[0]), "+r"(v[1])::"memory");
}
template <> __device__ __forceinline__ void tmem_wait_ld<4>(uint32_t (&v)[4])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(v[0]), "+r"(v[1]), "+r"(v[2]), "+r"(v[3])::"memory");
}

// ------------------------------------------------------------------ the sweep
// T: storage/arithmetic type.  R: rows (ROW) and columns (COL) per tile.
// E: hop entry type.  COL: which sweep.  LZ: Lanczos form.
// FOLD: the folded (eight-pass) Lanczos form.  It is an instantiation of its own because a kernel that merely CONTAINS
// tcgen05.alloc is scheduled differently (its CTAs hold the SM's allocation permit from launch): the
// nine-pass kernels have no tensor-memory instruction in them.
template <typename T, int R, typename E, bool COL, bool LZ, bool FOLD = false>
__global__ void __launch_bounds__(kGatherMaxThreads, 1)
gather_sweep_kernel(GatherArgs<T> A)
{
    static_assert(LZ || !FOLD, "the fold is a Lanczos form");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[32];
    __shared__ int flag;
    __shared__ __align__(8) uint64_t stage_bar;           // COL: bytes of the bulk-staged tile that have landed
    using PR = Pack<T, R>;
    using EB = typename BatchOf<E>::type;
    PR *Xs = reinterpret_cast<PR *>(smem_raw);            // [n_in_p + kZeroSlots]
    constexpr int kZeroSlots = 128 / (int)sizeof(PR);     // lanes served by one shared-memory wavefront
    const unsigned char *xs_bytes = smem_raw;

    const int nthr = (int)blockDim.x;                    // 1024, or less with several CTAs per SM (small sectors)
    const int64_t dd = A.dim_dn, du = A.dim_up;
    const int n_in = (int)A.in.dim;                       // contracted dimension
    const int n_in_p = (int)(COL ? A.du_p : A.dd_p);
    const int n_in_w = (n_in_p + 31) & ~31;               // whole warps run the gather loop (shuffles)
    const int64_t n_out_p = COL ? A.dd_p : A.du_p;
    const int64_t n_tiles = n_out_p / R;
    const E *__restrict__ ent = ent_ptr<E>(A.in);
    const int64_t ld = A.in.ld;
    const T tt = (T)A.t, UU = (T)A.U;

    // Folded form: line 4's "- b_{j+1} f_j" is applied by the ROW sweep, which has u_j in hand, as
    // z = (t H_dn + D) w - b_{j+1}^2 f_j  (so that c z = ... - b_{j+1} f_j), with b_{j+1}^2 = |q_j|^2 - a_j^2 known before
    // the sweep (|w|^2 itself only exists when the sweep ends; the recorded b_{j+1} is still that |w|).  The COL sweep
    // then reads w and z only.
    constexpr bool fold = FOLD;
    T ac = T(0), c = T(1), bcp = T(0), b2c = T(0);
    if (LZ) {
        if (A.S->stop) return;
        if (!COL) {
            ac = (T)(A.S->alpha * A.S->c_cur);            // line 6: w = q_j - a_j f_j, f_j = c_j u_j
            if (fold && A.S->started > 0) b2c = (T)((A.S->qnorm2 - A.S->alpha * A.S->alpha) * A.S->c_cur);
        } else {
            c = (T)A.S->c_cur;                            // f_{j+1} = c w
            if (!fold) bcp = (T)(A.S->beta * A.S->c_prev);    // b_{j+1} f_j = (b_{j+1} c_j) u_j
        }
    }
    if (!LZ && !COL && A.y_rowmajor && A.S) {
        // classic (three-kernel) Lanczos form on row-major vectors: y = c (t H_dn + D) x - b_j c_{j-1} y  (eq. 13, row half)
        if (A.S->stop) return;
        c = (T)A.S->c_cur;
        bcp = (T)(A.S->beta * A.S->c_prev);
    }
    if (threadIdx.x < kZeroSlots) {
        PR z;
#pragma unroll
        for (int r = 0; r < R; ++r) z.v[r] = T(0);
        Xs[n_in_p + threadIdx.x] = z;                     // zero slots, one per bank group (padding entries)
    }
    uint16_t *wsl_s = reinterpret_cast<uint16_t *>(smem_raw + (size_t)(n_in_p + kZeroSlots) * sizeof(PR));
    for (int i = threadIdx.x; i < n_in_w / 32; i += nthr) wsl_s[i] = A.in.wslots[i];   // slots per warp of positions
    double racc = 0.0;                                    // |w|^2 (ROW) or q.f (COL) partial
    double racc2 = 0.0;                                   // COL: |q|^2 partial
    const int64_t tile_bytes = (int64_t)n_in_p * (int64_t)sizeof(PR);
    // COL stages one contiguous block with no arithmetic on the way: a bulk copy when it is 16-byte granular
    const bool bulk_stage = COL && GS_TMA_STAGE && (tile_bytes % 16) == 0;
    unsigned stage_parity = 0;
    if (bulk_stage && threadIdx.x == 0) {
        mbar_init(&stage_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const int n_it = (n_in_w + nthr - 1) / nthr;                // gather iterations per tile
    // Position handled by this thread in iteration `it`: stripes of nthr positions, the warps of every other
    // stripe mirrored, so that with positions ordered by descending hop count all warps get equal work.
    const int wv = (int)(threadIdx.x >> 5), nwv = nthr >> 5, ln = (int)(threadIdx.x & 31);
    auto pos_of = [&](int it_) { return (it_ * nwv + ((it_ & 1) ? nwv - 1 - wv : wv)) * 32 + ln; };
    const int64_t pf_slice = ((tile_bytes + n_it - 1) / n_it + 15) / 16 * 16;       // bytes of the next tile requested per iteration
    const bool pf_ok = (tile_bytes % 16) == 0;            // bulk prefetches need 16-byte aligned addresses and sizes
    // buffers written in the other sweep's layout
    PR *outW = reinterpret_cast<PR *>(A.Wct);             // ROW: w (or x) in CT
    PR *outZ = reinterpret_cast<PR *>(COL ? A.Frt : A.Zct);   // ROW: z in CT;  COL/LZ: q in RT

    using LY = Layout<T, R>;
    constexpr int S = LY::S;
    // folded ROW sweep: this warp's columns of tensor memory, one piece per gather iteration
    constexpr int WPP = (int)sizeof(PR) / 4;              // 32-bit columns per piece
    __shared__ uint32_t tmem_base_s;
    uint32_t tcol = 0;
    constexpr bool park = !COL && fold;
    if (park) {
        if (wv == 0) tmem_alloc(&tmem_base_s, (uint32_t)A.fold_cols);
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        tcol = tmem_base_s + (((uint32_t)(wv & 3) * 32u) << 16) + (uint32_t)(wv >> 2) * (uint32_t)(n_it * WPP);
    }
    // Folded COL sweep: the first batch of a position's hop entries is what a thread waits for longest (it is requested
    // one short partial batch ahead; ncu: a third of the sweep's stall samples).  A thread gathers for the SAME positions
    // in every tile, so their first batches (16 bytes each, packed 16-bit entries) are parked in tensor memory once per
    // launch and come back with tcgen05.ld: no L2 round trip at the position switch, a third of the entry traffic gone.
    constexpr bool tment_k = COL && fold && sizeof(E) == 2;     // (instantiations that contain the tensor-memory path)
    const bool tment = tment_k && A.ent_cols > 0;
    constexpr int WPE = 4;                                      // 32-bit columns per parked batch
    if (tment_k) {
        if (tment) {
            if (wv == 0) tmem_alloc(&tmem_base_s, (uint32_t)A.ent_cols);
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncthreads();
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            tcol = tmem_base_s + (((uint32_t)(wv & 3) * 32u) << 16) + (uint32_t)(wv >> 2) * (uint32_t)(n_it * WPE);
            for (int it = 0; it < n_it; ++it) {
                const int i = pos_of(it);
                if (i >= n_in_w) continue;
                const EB e0 = load_batch(reinterpret_cast<const EB *>(ent) + i);
                uint32_t ew[WPE];
#pragma unroll
                for (int k = 0; k < WPE; ++k) ew[k] = e0.v[k];
                tmem_st<WPE>(tcol + (uint32_t)(it * WPE), ew);
            }
            tmem_wait_st();
        } else if (wv == 0) {
            // (a CTA of a kernel that contains tcgen05.alloc holds the SM's allocation permit until it gives it up)
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
    }
    // first batch of the entries of this thread's position in gather iteration it_ (requested; see first_batch_ready)
    auto first_batch = [&](int it_) {
        EB e;
        if constexpr (tment_k) {
            if (tment) {
                uint32_t ew[WPE] = {0u, 0u, 0u, 0u};
                if (it_ < n_it) tmem_ld<WPE>(tcol + (uint32_t)(it_ * WPE), ew);
#pragma unroll
                for (int k = 0; k < WPE; ++k) e.v[k] = ew[k];
                return e;
            }
        }
        return load_batch(reinterpret_cast<const EB *>(ent) + min(pos_of(it_), n_in_w - 1));
    };
    auto first_batch_ready = [&](EB &e) {
        if constexpr (tment_k) {
            if (tment) {
                uint32_t ew[WPE];
#pragma unroll
                for (int k = 0; k < WPE; ++k) ew[k] = e.v[k];
                tmem_wait_ld<WPE>(ew);
#pragma unroll
                for (int k = 0; k < WPE; ++k) e.v[k] = ew[k];
            }
        }
    };
    // piece of position i of the current tile
    auto poff = [&](int i) { return S == 1 ? (int64_t)i : (int64_t)(i / R) * (S * R) + i % R; };

    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int64_t o0 = tile * R;
        const int64_t tbase = LY::piece(tile, 0, n_in_p);
        __syncthreads();                                  // gathers of the previous tile are done
        // ---- stage the tile
        if (COL || LZ) {
            // tile-major layouts: the pieces are already the interleaved shared-memory image
            const PR *src = reinterpret_cast<const PR *>(COL ? A.Wct : A.Qrt) + tbase;
            if (park) {
                // same thread <-> position map as the gather, so that the piece of u_j parked here is this thread's
                // own in the epilogue (whole warps: the tensor-memory accesses are warp-collective)
                const PR *fsrc = reinterpret_cast<const PR *>(A.Frt) + tbase;
                PR *wdst = reinterpret_cast<PR *>(A.Qrt) + tbase;
                for (int it0 = 0; it0 < n_it; it0 += GS_PARK_UNROLL) {
                    PR v[GS_PARK_UNROLL], f[GS_PARK_UNROLL];
#pragma unroll
                    for (int u = 0; u < GS_PARK_UNROLL; ++u) {
                        const int i = pos_of(it0 + u);
#pragma unroll
                        for (int r = 0; r < R; ++r) v[u].v[r] = f[u].v[r] = T(0);
                        if (it0 + u < n_it && i < n_in_p) { v[u] = ld_stage(src + poff(i)); f[u] = ld_stage(fsrc + poff(i)); }
                    }
#pragma unroll
                    for (int u = 0; u < GS_PARK_UNROLL; ++u) {
                        const int it = it0 + u;
                        const int i = pos_of(it);
                        if (it >= n_it || i >= n_in_w) continue;
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            v[u].v[r] = v[u].v[r] - ac * f[u].v[r];
                            racc += (double)v[u].v[r] * (double)v[u].v[r];
                        }
                        if (i < n_in_p) {
                            st_once<1>(wdst + poff(i), v[u]);
                            Xs[i] = v[u];
                        }
                        uint32_t fw[WPP];
                        memcpy(fw, &f[u], sizeof(PR));
                        tmem_st<WPP>(tcol + (uint32_t)(it * WPP), fw);
                    }
                }
                tmem_wait_st();
            } else if (!COL) {
                const PR *fsrc = reinterpret_cast<const PR *>(A.Frt) + tbase;
                PR *wdst = reinterpret_cast<PR *>(A.Qrt) + tbase;
                // loads of kStageUnroll pieces are issued before the first store (w overwrites q in place)
                for (int i0 = threadIdx.x; i0 < n_in_p; i0 += kStageUnroll * nthr) {
                    PR v[kStageUnroll], f[kStageUnroll];
#pragma unroll
                    for (int u = 0; u < kStageUnroll; ++u) {
                        const int i = i0 + u * nthr;
                        if (i < n_in_p) { v[u] = ld_once<1>(src + poff(i)); f[u] = ld_once<1>(fsrc + poff(i)); }
                    }
#pragma unroll
                    for (int u = 0; u < kStageUnroll; ++u) {
                        const int i = i0 + u * nthr;
                        if (i < n_in_p) {
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                v[u].v[r] = v[u].v[r] - ac * f[u].v[r];
                                racc += (double)v[u].v[r] * (double)v[u].v[r];
                            }
                            st_once<1>(wdst + poff(i), v[u]);
                            Xs[i] = v[u];
                        }
                    }
                }
            } else if (bulk_stage) {
                // (the barrier above ordered the previous tile's shared-memory reads; the proxy fence orders them
                // against the asynchronous writes that follow)
                if (threadIdx.x == 0) {
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    mbar_expect_tx(&stage_bar, (unsigned)tile_bytes);
                    constexpr int64_t kChunk = 32768;
                    for (int64_t off = 0; off < tile_bytes; off += kChunk)
                        bulk_g2s(smem_raw + off, reinterpret_cast<const char *>(src) + off, (unsigned)min(kChunk, tile_bytes - off), &stage_bar);
                }
                mbar_wait(&stage_bar, stage_parity);
                stage_parity ^= 1u;
            } else {
                for (int i0 = threadIdx.x; i0 < n_in_p; i0 += kStageUnroll * nthr) {
                    PR v[kStageUnroll];
#pragma unroll
                    for (int u = 0; u < kStageUnroll; ++u) {
                        const int i = i0 + u * nthr;
                        if (i < n_in_p) v[u] = ld_once<2>(src + poff(i));
                    }
#pragma unroll
                    for (int u = 0; u < kStageUnroll; ++u) {
                        const int i = i0 + u * nthr;
                        if (i < n_in_p) Xs[i] = v[u];
                    }
                }
            }
        } else {
            // ROW sweep of hubbard_apply: x is the caller's row-major array
            int vw = R;                                   // columns per vector load: rows must stay 16-byte aligned
            while (vw > 1 && ((dd % vw) != 0 || (sizeof(T) * vw > 16))) vw >>= 1;
            if (R >= 4 && vw == 4) stage_rowmajor<T, R, (R >= 4 ? 4 : 1)>(A.x, Xs, o0, du, dd, n_in, n_in_p, nthr);
            else if (R >= 2 && vw >= 2) stage_rowmajor<T, R, (R >= 2 ? 2 : 1)>(A.x, Xs, o0, du, dd, n_in, n_in_p, nthr);
            else stage_rowmajor<T, R, 1>(A.x, Xs, o0, du, dd, n_in, n_in_p, nthr);
        }
        __syncthreads();

        // ---- gather: one thread per contracted index i, R outputs each
        uint32_t so[R];
        if (!COL) {
#pragma unroll
            for (int r = 0; r < R; ++r) so[r] = (o0 + r < du) ? A.st_out[o0 + r] : 0u;
        }
        // every position has >= 1 (padding) batch; the table has n_in_w batches per plane, a block may have more threads
        EB pk = first_batch(0);
        for (int it = 0; it < n_it; ++it) {
            const int i = pos_of(it);
            first_batch_ready(pk);                        // (before the skip: a tensor-memory load must not stay pending)
            if (i >= n_in_w) continue;                    // whole warps: a partly filled last stripe (the last iteration only)
            const bool valid = i < n_in;
            const bool inpad = i < n_in_p;
            const int n = (int)wsl_s[i >> 5];                // warp-uniform, >= 1
            // operands of the epilogue: requested now, used after the gather
            uint32_t sd = 0u;
            PR z, f;
#pragma unroll
            for (int r = 0; r < R; ++r) z.v[r] = f.v[r] = T(0);
            uint32_t fw[WPP];
#if GS_HOIST
            if (!COL) {
                if (valid) sd = A.in.st[i];
                if (park && !GS_FOLD_LATE) tmem_ld<WPP>(tcol + (uint32_t)(it * WPP), fw);
            } else if (inpad) {
                z = ld_once<(sizeof(T) == 4 ? 4 : 8)>(reinterpret_cast<const PR *>(A.Zct) + tbase + poff(i));
                if (LZ && !fold) f = ld_once<(sizeof(T) == 4 ? 4 : 8)>(reinterpret_cast<const PR *>(A.Fct) + tbase + poff(i));
            }
#endif
            // keep DRAM busy during the gather: a slice of the next tile's inputs goes to L2 every iteration
#if GS_L2PF
            // (the S tiles of a super-tile share one contiguous region of S * tile_bytes: each of their CTAs
            // requests the S-th part of it that has its own number)
            if ((COL || LZ) && pf_ok && tile + gridDim.x < n_tiles) {
                const int64_t off = (int64_t)it * pf_slice + (int64_t)threadIdx.x * 2048;
                if (threadIdx.x * 2048 < pf_slice && off < tile_bytes) {
                    const unsigned nb = (unsigned)min((int64_t)2048, min(pf_slice - (int64_t)threadIdx.x * 2048, tile_bytes - off));
                    const int64_t tn = tile + gridDim.x;
                    const int64_t region = LY::piece(tn - tn % S, 0, n_in_p) + (tn % S) * (int64_t)n_in_p;    // in pieces
                    const char *p0 = reinterpret_cast<const char *>(reinterpret_cast<const PR *>(COL ? A.Wct : A.Qrt) + region) + off;
                    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p0), "r"(nb) : "memory");
                    if (!COL) {
                        const char *p1 = reinterpret_cast<const char *>(reinterpret_cast<const PR *>(A.Frt) + region) + off;
                        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p1), "r"(nb) : "memory");
                    }
                }
            }
#endif
            T acc[R];
#pragma unroll
            for (int r = 0; r < R; ++r) acc[r] = T(0);
            // one batch of hop entries is always in flight: the next batch of this state, or the first
            // batch of this thread's next state
            const EB *ep = reinterpret_cast<const EB *>(ent) + i;
            const int nb = (n + kGatherBatch - 1) / kGatherBatch;
            // the first batch of the NEXT position: the fp32 ROW sweep requests it a whole position ahead, the others just
            // before this position's last batch (the folded COL sweep from tensor memory)
            EB nxtpos;
            // (measured on C4: ROW fp32 0.989 -> 0.966 ms, fp64 1.806 -> 1.826 ms; the COL sweeps have no registers for it)
            constexpr bool early_first = GS_EARLY_FIRST && !COL && sizeof(T) == 4;
            if (early_first) nxtpos = first_batch(it + 1);
            int b = 0;
            // (the nine-pass COL sweep, which holds two epilogue operands over the gather, spills 8 bytes for this and is still
            // faster with it: C3 0.173 against 0.188 ms)
            for (; b + 2 < nb; b += 2) {                  // two full batches per trip: no register copies between them
                ep += ld;
                const EB n1 = load_batch(ep);
                hop_batch_n<T, R>(xs_bytes, pk, kGatherBatch, acc);
                ep += ld;
                pk = load_batch(ep);
                hop_batch_n<T, R>(xs_bytes, n1, kGatherBatch, acc);
            }
            for (; b + 1 < nb; ++b) {
                ep += ld;
                const EB nxt = load_batch(ep);
                hop_batch_n<T, R>(xs_bytes, pk, kGatherBatch, acc);
                pk = nxt;
            }
            {
                if (!early_first) nxtpos = first_batch(it + 1);
                hop_batch_n<T, R>(xs_bytes, pk, n - (nb - 1) * kGatherBatch, acc);    // 1..8 entries, warp-uniform
                pk = nxtpos;
            }
            PR xi;
#pragma unroll
            for (int r = 0; r < R; ++r) xi.v[r] = T(0);
            if (inpad) xi = Xs[i];
#if !GS_HOIST
            if (!COL) {
                if (valid) sd = A.in.st[i];
                if (park && !GS_FOLD_LATE) tmem_ld<WPP>(tcol + (uint32_t)(it * WPP), fw);
            } else if (inpad) {
                z = ld_once<(sizeof(T) == 4 ? 4 : 8)>(reinterpret_cast<const PR *>(A.Zct) + tbase + poff(i));
                if (LZ && !fold) f = ld_once<(sizeof(T) == 4 ? 4 : 8)>(reinterpret_cast<const PR *>(A.Fct) + tbase + poff(i));
            }
#endif
            const int q = i % R;
            // this lane's piece in the other layout (R adjacent lanes: one 32/64-byte sector)
            const int64_t oidx = LY::piece(i / R, o0 + q, n_out_p);
            if (!COL) {
                // Algorithm 4: on-the-fly diagonal
                T h[R];
#pragma unroll
                for (int r = 0; r < R; ++r) h[r] = tt * acc[r] + UU * (T)__popc(so[r] & sd) * xi.v[r];
                if (park) {
                    if (GS_FOLD_LATE) tmem_ld<WPP>(tcol + (uint32_t)(it * WPP), fw);
                    tmem_wait_ld<WPP>(fw);
                    memcpy(&f, fw, sizeof(PR));
#pragma unroll
                    for (int r = 0; r < R; ++r) h[r] -= b2c * f.v[r];          // - b_{j+1}^2 f_j (line 4, eq. 13)
                }
                if (!LZ && A.y_rowmajor) {
                    // hubbard_apply, hybrid form: y = (t H_dn + D) x in the caller's row-major layout
                    // (coalesced over i for each of the R rows); the strip sweep adds the up term
                    if (valid) {
#pragma unroll
                        for (int r = 0; r < R; ++r)
                            if (o0 + r < du) {
                                const int64_t J = (o0 + r) * dd + i;
                                A.y[J] = A.S ? c * h[r] - bcp * A.y[J] : h[r];
                            }
                    }
                } else {
                    const PR wt = block_transpose<T, R>(xi.v, q);
                    const PR zt = block_transpose<T, R>(h, q);
                    if (inpad) {
                        st_once<2>(outW + oidx, wt);
                        st_once<2>(outZ + oidx, zt);
                    }
                }
            } else {
                if (LZ) {
                    T qv[R];
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        qv[r] = c * (tt * acc[r] + z.v[r]) - bcp * f.v[r];      // line 4 + eq. 13
                        racc += (double)qv[r] * (double)(c * xi.v[r]);          // line 5
                        if (fold) racc2 += (double)qv[r] * (double)qv[r];
                    }
                    const PR qt = block_transpose<T, R>(qv, q);
                    if (inpad) st_once<4>(outZ + oidx, qt);
                } else if (valid) {
                    // hubbard_apply: y is the caller's row-major array; one write per element
                    T *yr = A.y + (int64_t)i * dd + o0;
#pragma unroll
                    for (int r = 0; r < R; ++r)
                        if (o0 + r < dd) yr[r] = tt * acc[r] + z.v[r];
                }
            }
        }
    }

    if (park || tment) {
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (wv == 0) tmem_dealloc(tmem_base_s, (uint32_t)(park ? A.fold_cols : A.ent_cols));
    }
    if (LZ) {
        const double sblk = block_sum(racc, red);
        if (COL && fold) {
            // second partial of the block, published by the same ticket (thread 0 writes both before its fence)
            const double sblk2 = block_sum(racc2, red);
            if (threadIdx.x == 0) A.partials[gridDim.x + blockIdx.x] = sblk2;
        }
        if (publish_and_check_last(sblk, A.partials, blockIdx.x, gridDim.x, &A.S->ticket, &flag)) {
            const double tot = sum_partials(A.partials, gridDim.x, red);
            if (!COL) {
                if (threadIdx.x == 0) lanczos_rotate(A.S, tot, A.alpha_out, A.beta_out);
            } else {
                const double tot2 = fold ? sum_partials(A.partials + gridDim.x, gridDim.x, red) : 0.0;
                if (threadIdx.x == 0) {
                    A.S->alpha = tot;
                    A.S->qnorm2 = tot2;
                    A.S->ticket = 0;
                }
            }
        }
    }
}

// Start of a run: the caller's row-major start vector (basis order of PAPER.md:63-71) into the RT layout in
// the internal order of both spins (zero padding included).  One thread per 16-byte piece.
template <typename T, int R>
__global__ void __launch_bounds__(256)
to_rt_kernel(const T *__restrict__ x, T *__restrict__ rt, int64_t du, int64_t dd, int64_t du_p, int64_t dd_p,
             const int32_t *__restrict__ perm_up, const int32_t *__restrict__ perm_dn)
{
    using PR = Pack<T, R>;
    constexpr int S = Layout<T, R>::S;
    const int64_t n = du_p / R * dd_p;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
        // piece p of the RT layout -> (row tile, column position)
        const int64_t t1 = p / R, t2 = t1 / S;
        const int64_t tile = (t2 / (dd_p / R)) * S + t1 % S, bp = (t2 % (dd_p / R)) * R + p % R;
        const int64_t b = (bp < dd) ? perm_dn[bp] : -1;
        PR v;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int64_t ap = tile * R + r;
            const int64_t a = (ap < du) ? perm_up[ap] : -1;
            v.v[r] = (a >= 0 && b >= 0) ? x[a * dd + b] : T(0);
        }
        reinterpret_cast<PR *>(rt)[p] = v;
    }
}

// Closing sweep of a run: b_{m+1} = |q_m - a_m f_m| (Algorithm 1 lines 6-7) for
// the last iteration, nothing written but the scalars.
template <typename T>
__global__ void __launch_bounds__(512)
lanczos_final_norm_kernel(const T *__restrict__ Q, const T *__restrict__ F, int64_t dim, LanczosScalars *S,
                          double *partials, double *alpha_out, double *beta_out)
{
    __shared__ double red[32];
    __shared__ int flag;
    if (S->stop) return;
    const T ac = (T)(S->alpha * S->c_cur);
    double acc = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < dim; i += (int64_t)gridDim.x * blockDim.x) {
        const T v = Q[i] - ac * F[i];
        acc += (double)v * (double)v;
    }
    const double sblk = block_sum(acc, red);
    if (publish_and_check_last(sblk, partials, blockIdx.x, gridDim.x, &S->ticket, &flag)) {
        const double tot = sum_partials(partials, gridDim.x, red);
        if (threadIdx.x == 0) lanczos_rotate(S, tot, alpha_out, beta_out);
    }
}

// The RT layout (internal order) back into the caller's row-major layout (ground-state vector).
template <typename T, int R>
__global__ void __launch_bounds__(256)
from_rt_kernel(const T *__restrict__ rt, T *__restrict__ x, int64_t du, int64_t dd, int64_t du_p, int64_t dd_p,
               const int32_t *__restrict__ perm_up, const int32_t *__restrict__ perm_dn)
{
    using PR = Pack<T, R>;
    constexpr int S = Layout<T, R>::S;
    const int64_t n = du_p / R * dd_p;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
        const int64_t t1 = p / R, t2 = t1 / S;
        const int64_t tile = (t2 / (dd_p / R)) * S + t1 % S, bp = (t2 % (dd_p / R)) * R + p % R;
        const int64_t b = (bp < dd) ? perm_dn[bp] : -1;
        const PR v = reinterpret_cast<const PR *>(rt)[p];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int64_t ap = tile * R + r;
            const int64_t a = (ap < du) ? perm_up[ap] : -1;
            if (a >= 0 && b >= 0) x[a * dd + b] = v.v[r];
        }
    }
}

__global__ void lanczos_scalars_init_kernel(LanczosScalars *S, double tau)
{
    S->c_cur = 0.0; S->c_prev = 0.0; S->beta = 0.0; S->alpha = 0.0; S->amax = 0.0; S->tau = tau;
    S->j = 0; S->stop = 0; S->ticket = 0; S->started = 0; S->qnorm2 = 0.0;
}

}  // namespace hub
