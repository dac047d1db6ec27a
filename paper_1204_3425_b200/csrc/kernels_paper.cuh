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
};

constexpr int kPaperThreads = 256;

template <typename T, bool LANCZOS>
__global__ void __launch_bounds__(kPaperThreads)
hv_paper_kernel(DevModel M, SweepArgs<T> A)
{
    extern __shared__ uint32_t s_up[];   // w_up entries of the current up row
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

    for (int64_t a = blockIdx.y; a < M.dim_up; a += gridDim.y) {
        const int nup = M.up_cnt[a];
        __syncthreads();
        for (int k = threadIdx.x; k < nup; k += blockDim.x) s_up[k] = M.up_ent[a * M.w_up + k];
        __syncthreads();
        if (!active) continue;
        const T *xa = A.x + a * M.dim_dn;
        T sum = T(0);
        // Algorithm 2: (H_up (x) I) x — whole-row, coalesced reads
        for (int k = 0; k < nup; ++k) {
            uint32_t e = s_up[k];
            sum += signed_by(e, A.x[(int64_t)(e >> 1) * M.dim_dn + b]);
        }
        // Algorithm 3: (I (x) H_dn) x — gather inside row a
        for (int k = 0; k < ndn; ++k) {
            uint32_t e = M.dn_ent32[(int64_t)k * M.ld_dn + b];
            sum += signed_by(e, xa[e >> 1]);
        }
        // Algorithm 4: on-the-fly diagonal
        const T xv = xa[b];
        T h = tt * sum + UU * (T)__popc(M.st_up[a] & sdn) * xv;
        if (LANCZOS) {
            T *ya = A.y + a * M.dim_dn;
            T q = c_cur * h - bc * ya[b];
            ya[b] = q;
            acc += (double)q * (double)(c_cur * xv);
        } else {
            A.y[a * M.dim_dn + b] = h;
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
