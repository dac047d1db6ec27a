// Variant TWOSWEEP: H v in two device-wide sweeps chosen for B200's memory
// system:
//
//   row sweep    y = c (t (I (x) H_dn) x + D o x) - bc y      eq. 16 + Algorithm 4
//                (PAPER.md:281-317,325-334).  A group of R whole rows of V is
//                staged in shared memory; every gather of the down term is a
//                shared-memory read; the hop entries of a column are read once
//                per group and reused for its R rows.
//   strip sweep  y += c t (H_up (x) I) x, a_j = <y, c x>        eq. 15
//                (PAPER.md:238-277).  Work is ordered by column strip so that
//                V[:, strip] stays resident in L2 while its ~18 re-reads per
//                element happen; DRAM sees each element of x once per sweep.
//
// In the Lanczos form (c = c_cur, bc = b_j c_prev) y is f_{j-1}'s storage and
// becomes q_j (eq. 13); the strip sweep also reduces
// a_j = q_j . f_j (Algorithm 1 line 5).
#pragma once
#include "kernels_common.cuh"
#include "kernels_paper.cuh"

namespace hub {

constexpr int kRowThreads = 1024;
constexpr int kStripThreads = 256;

template <typename T, int VW> struct VecOf;
template <> struct VecOf<float, 1>  { using type = float; };
template <> struct VecOf<float, 2>  { using type = float2; };
template <> struct VecOf<float, 4>  { using type = float4; };
template <> struct VecOf<double, 1> { using type = double; };
template <> struct VecOf<double, 2> { using type = double2; };

// ---------------------------------------------------------------- row sweep
// E: hop entry type (uint16_t compact / uint32_t).  R: rows per group.
template <typename T, typename E, int R, bool LANCZOS>
__global__ void __launch_bounds__(kRowThreads, 1)
row_sweep_kernel(DevModel M, SweepArgs<T> A, const E *__restrict__ dn_ent)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *s = reinterpret_cast<T *>(smem_raw);
    constexpr int N = 16 / sizeof(T);
    using V = typename VecOf<T, N>::type;

    T c_cur = T(1), bc = T(0);
    if (LANCZOS) {
        if (A.S->stop) return;
        c_cur = (T)A.S->c_cur;
        bc = (T)(A.S->beta * A.S->c_prev);
    }
    const T ct = c_cur * (T)M.t, cU = c_cur * (T)M.U;
    const int64_t dd = M.dim_dn;
    const int64_t n_groups = (M.dim_up + R - 1) / R;

    for (int64_t g = blockIdx.x; g < n_groups; g += gridDim.x) {
        const int64_t a0 = g * R;
        const int nr = (int)min((int64_t)R, M.dim_up - a0);
        const int64_t e0 = a0 * dd, cnt = (int64_t)nr * dd;
        const int phase = (int)(e0 % N);          // keep the global 16-byte phase in shared memory
        const T *src = A.x + e0;
        T *dst = s + phase;
        __syncthreads();                           // previous group's gathers are done
        const int64_t head = min(cnt, (int64_t)((N - phase) % N));
        const int64_t nvec = (cnt - head) / N;
        for (int64_t i = threadIdx.x; i < head; i += blockDim.x) dst[i] = src[i];
        {
            const V *sv = reinterpret_cast<const V *>(src + head);
            V *dv = reinterpret_cast<V *>(dst + head);
            for (int64_t i = threadIdx.x; i < nvec; i += blockDim.x) dv[i] = __ldcs(sv + i);
        }
        for (int64_t i = head + nvec * N + threadIdx.x; i < cnt; i += blockDim.x) dst[i] = src[i];
        __syncthreads();

        for (int64_t b = threadIdx.x; b < dd; b += blockDim.x) {
            const int n = M.dn_cnt[b];
            const uint32_t sdn = M.st_dn[b];
            T sum[R];
#pragma unroll
            for (int r = 0; r < R; ++r) sum[r] = T(0);
            const E *ep = dn_ent + b;
            for (int k = 0; k < n; ++k) {
                const uint32_t e = ep[(int64_t)k * M.ld_dn];
                const T *p = dst + (e >> 1);
#pragma unroll
                for (int r = 0; r < R; ++r) sum[r] += signed_by(e, p[(int64_t)r * dd]);
            }
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if (r < nr) {
                    const int64_t J = e0 + (int64_t)r * dd + b;
                    const T xv = dst[(int64_t)r * dd + b];
                    T h = ct * sum[r] + cU * (T)__popc(M.st_up[a0 + r] & sdn) * xv;
                    if (LANCZOS) h -= bc * A.y[J];
                    A.y[J] = h;
                }
            }
        }
    }
}

// Row sweep without staging, for rows that do not fit in shared memory: the
// gathers go through L1/L2 (same arithmetic as Algorithm 3).
template <typename T, typename E, bool LANCZOS>
__global__ void __launch_bounds__(kPaperThreads)
row_sweep_direct_kernel(DevModel M, SweepArgs<T> A, const E *__restrict__ dn_ent)
{
    T c_cur = T(1), bc = T(0);
    if (LANCZOS) {
        if (A.S->stop) return;
        c_cur = (T)A.S->c_cur;
        bc = (T)(A.S->beta * A.S->c_prev);
    }
    const T ct = c_cur * (T)M.t, cU = c_cur * (T)M.U;
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= M.dim_dn) return;
    const int n = M.dn_cnt[b];
    const uint32_t sdn = M.st_dn[b];
    for (int64_t a = blockIdx.y; a < M.dim_up; a += gridDim.y) {
        const T *xa = A.x + a * M.dim_dn;
        T sum = T(0);
        for (int k = 0; k < n; ++k) {
            const uint32_t e = dn_ent[(int64_t)k * M.ld_dn + b];
            sum += signed_by(e, __ldg(xa + (e >> 1)));
        }
        const int64_t J = a * M.dim_dn + b;
        T h = ct * sum + cU * (T)__popc(M.st_up[a] & sdn) * xa[b];
        if (LANCZOS) h -= bc * A.y[J];
        A.y[J] = h;
    }
}

// -------------------------------------------------------------- strip sweep
struct StripPlan {
    int64_t W;        // strip width in elements (multiple of the vector width)
    int64_t n_strips;
    int RB;           // rows per block
    int64_t bps;      // blocks per strip = ceil(dim_up / RB)
};

template <typename T, int VW, bool LANCZOS>
__global__ void __launch_bounds__(kStripThreads)
strip_sweep_kernel(DevModel M, SweepArgs<T> A, StripPlan P)
{
    extern __shared__ uint32_t s_ent[];     // [RB][w_up] entries, then [RB] counts
    __shared__ double red[32];
    __shared__ int flag;
    using V = typename VecOf<T, VW>::type;

    T c_cur = T(1);
    if (LANCZOS) {
        if (A.S->stop) return;
        c_cur = (T)A.S->c_cur;
    }
    const T ct = c_cur * (T)M.t;
    const int64_t strip = blockIdx.x / P.bps, rb = blockIdx.x % P.bps;
    const int64_t c0 = strip * P.W, c1 = min(M.dim_dn, c0 + P.W);
    const int64_t r0 = rb * P.RB;
    const int nrow = (int)min((int64_t)P.RB, M.dim_up - r0);
    int *s_cnt = reinterpret_cast<int *>(s_ent + (size_t)P.RB * M.w_up);

    for (int i = threadIdx.x; i < nrow * M.w_up; i += blockDim.x) s_ent[i] = M.up_ent[r0 * M.w_up + i];
    for (int i = threadIdx.x; i < nrow; i += blockDim.x) s_cnt[i] = M.up_cnt[r0 + i];
    __syncthreads();

    const int vpr = (int)((c1 - c0) / VW);          // vectors per row inside the strip (c1-c0 is a multiple of VW)
    const int items = nrow * vpr;
    double acc = 0.0;
    for (int it = threadIdx.x; it < items; it += blockDim.x) {
        const int rl = it / vpr, vi = it - rl * vpr;
        const int64_t c = c0 + (int64_t)vi * VW;
        const uint32_t *ent = s_ent + rl * M.w_up;
        const int n = s_cnt[rl];
        T sum[VW];
#pragma unroll
        for (int q = 0; q < VW; ++q) sum[q] = T(0);
        for (int k = 0; k < n; ++k) {
            const uint32_t e = ent[k];
            V v = __ldg(reinterpret_cast<const V *>(A.x + (int64_t)(e >> 1) * M.dim_dn + c));
            const T *ve = reinterpret_cast<const T *>(&v);
#pragma unroll
            for (int q = 0; q < VW; ++q) sum[q] += signed_by(e, ve[q]);
        }
        const int64_t J = (r0 + rl) * M.dim_dn + c;
        V yv = __ldcs(reinterpret_cast<const V *>(A.y + J));
        T *ye = reinterpret_cast<T *>(&yv);
#pragma unroll
        for (int q = 0; q < VW; ++q) ye[q] += ct * sum[q];
        __stcs(reinterpret_cast<V *>(A.y + J), yv);
        if (LANCZOS) {
            V xv = __ldg(reinterpret_cast<const V *>(A.x + J));
            const T *xe = reinterpret_cast<const T *>(&xv);
#pragma unroll
            for (int q = 0; q < VW; ++q) acc += (double)ye[q] * (double)(c_cur * xe[q]);
        }
    }
    if (LANCZOS) {
        double sblk = block_sum(acc, red);
        if (publish_and_check_last(sblk, A.partials, blockIdx.x, gridDim.x, &A.S->ticket, &flag)) {
            double alpha = sum_partials(A.partials, gridDim.x, red);
            if (threadIdx.x == 0) {
                A.S->alpha = alpha;
                A.S->ticket = 0;
            }
        }
    }
}

}  // namespace hub
