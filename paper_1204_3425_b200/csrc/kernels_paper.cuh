// Variant PAPER: Algorithms 2-4 of the paper restated for sm_100a
// (PAPER.md:238-317): one thread per element of the result, the ELL row of
// H_up staged in shared memory, the ELL column of H_dn read coalesced from
// global memory, the diagonal generated on the fly, ONE write of the sum
// (PAPER.md:236,336).  Kept as the in-box "prior art on the same GPU"
// comparator and as the path for sectors the tuned kernels do not cover.
//
// LANCZOS = true fuses line 4 and line 5 of Algorithm 1
// with eq. 13: q = H f_j - b_j f_{j-1} is written over
// f_{j-1} and a_j = q.f_j is reduced in the same sweep.
#pragma once
#include "kernels_common.cuh"

namespace hub {

template <typename T>
struct SweepArgs {
    const T *x;            // u_cur  (f_j = c_cur * u_cur), or x of hubbard_apply
    T *y;                  // u_prev in / q out (Lanczos), or y of hubbard_apply
    LanczosScalars *S;     // null for plain apply
    double *partials;
    // row-sharded H v (hubbard_apply_rows): rows [a_begin, a_end) of the result from the FULL x; y holds only those
    // rows (row a at (a - a_begin) * dim_dn).  a_end == 0 means all rows.
    int64_t a_begin = 0, a_end = 0;
};

constexpr int kPaperThreads = 256;

// SUB = sub-vectors (rows of V) per block = elements per thread.  SUB = 1 is
// Algorithms 2-4 as printed; SUB = 4 is the paper's own tuning (PAPER.md:338:
// "four elements per thread, i.e. four subvectors per block"): the block stages
// the ELL rows of H_up of its SUB sub-vectors ("increases register and shared
// memory usage") and each down-hop entry Ax/Aj[i * dimDn + id] is loaded once
// for the SUB elements a thread owns.
template <typename T, bool LANCZOS, int SUB>
__global__ void __launch_bounds__(kPaperThreads)
hv_paper_kernel(DevModel M, SweepArgs<T> A)
{
    extern __shared__ uint32_t s_up[];   // SUB x w_up entries: the up rows of the block's sub-vectors
    __shared__ double red[32];
    __shared__ int flag;

    T c_cur = T(1), bc = T(0);
    if (LANCZOS) {
        if (A.S->stop) return;
        c_cur = (T)A.S->c_cur;
        bc = (T)(A.S->beta * A.S->c_prev);
    }
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = b < M.dim_dn;
    const T tt = (T)M.t, UU = (T)M.U;
    double acc = 0.0;

    // down-hop entries of column b do not depend on the row: keep the count
    const int ndn = active ? M.dn_cnt[b] : 0;
    const uint32_t sdn = active ? M.st_dn[b] : 0u;

    const int64_t a_end = A.a_end > 0 ? A.a_end : M.dim_up;
    T *const yb = A.y - A.a_begin * M.dim_dn;            // row a of the result at yb + a * dim_dn
    for (int64_t a0 = A.a_begin + (int64_t)blockIdx.y * SUB; a0 < a_end; a0 += (int64_t)gridDim.y * SUB) {
        int nup[SUB];
#pragma unroll
        for (int r = 0; r < SUB; ++r) nup[r] = (a0 + r < a_end) ? M.up_cnt[a0 + r] : 0;
        __syncthreads();
#pragma unroll
        for (int r = 0; r < SUB; ++r)
            for (int k = threadIdx.x; k < nup[r]; k += blockDim.x) s_up[r * M.w_up + k] = M.up_ent[(a0 + r) * M.w_up + k];
        __syncthreads();
        if (!active) continue;
        T sum[SUB];
        // Algorithm 2: (H_up (x) I) x — whole-row, coalesced reads
#pragma unroll
        for (int r = 0; r < SUB; ++r) {
            sum[r] = T(0);
            for (int k = 0; k < nup[r]; ++k) {
                uint32_t e = s_up[r * M.w_up + k];
                sum[r] += signed_by(e, A.x[(int64_t)(e >> 1) * M.dim_dn + b]);
            }
        }
        // Algorithm 3: (I (x) H_dn) x — gather inside each of the SUB rows, one entry load for all of them
        for (int k = 0; k < ndn; ++k) {
            uint32_t e = M.dn_ent32[(int64_t)k * M.ld_dn + b];
#pragma unroll
            for (int r = 0; r < SUB; ++r)
                if (a0 + r < a_end) sum[r] += signed_by(e, A.x[(a0 + r) * M.dim_dn + (e >> 1)]);
        }
#pragma unroll
        for (int r = 0; r < SUB; ++r) {
            const int64_t a = a0 + r;
            if (a >= a_end) break;
            // Algorithm 4: on-the-fly diagonal
            const T xv = A.x[a * M.dim_dn + b];
            T h = tt * sum[r] + UU * (T)__popc(M.st_up[a] & sdn) * xv;
            if (LANCZOS) {
                T *ya = yb + a * M.dim_dn;
                T q = c_cur * h - bc * ya[b];
                ya[b] = q;
                acc += (double)q * (double)(c_cur * xv);
            } else {
                yb[a * M.dim_dn + b] = h;
            }
        }
    }
    if (LANCZOS) {
        double s = block_sum(acc, red);
        unsigned nb = gridDim.x * gridDim.y;
        int64_t slot = (int64_t)blockIdx.y * gridDim.x + blockIdx.x;
        if (publish_and_check_last(s, A.partials, slot, nb, &A.S->ticket, &flag)) {
            double alpha = sum_partials(A.partials, nb, red);
            if (threadIdx.x == 0) {
                A.S->alpha = alpha;
                A.S->ticket = 0;
            }
        }
    }
}

}  // namespace hub
