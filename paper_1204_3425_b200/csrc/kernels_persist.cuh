// Variant PERSIST: the whole Lanczos loop of a SMALL sector in one cooperative
// kernel (SURVEY.md hard part H5: configurations 1-2 are launch-latency
// problems; their vectors are L2-resident).  Algorithms 2-4 per element as in
// variant PAPER, Algorithm 1 with eq. 13 around them
// (PAPER.md:116-164); the two global reductions of an iteration (lines 5 and 7)
// are grid-wide barriers instead of kernel boundaries: per-block partials,
// grid.sync(), every block sums the partials in index order (deterministic and
// identical in all blocks, so the scalars live in registers).
#pragma once
#include <cooperative_groups.h>

#include "kernels_common.cuh"

namespace hub {

constexpr int kPersistThreads = 512;

template <typename T>
struct PersistArgs {
    T *vec0, *vec1;          // vec[j & 1] = u_{j+1} (f = c_cur u), vec[(j + 1) & 1] = u_j -> q -> w
    LanczosScalars *S;       // state between calls (c_cur, c_prev, beta, amax, j, stop)
    double *part_a, *part_b; // gridDim.x doubles each
    double *alpha_out, *beta_out;
    int j0, j1;
    const double *ycoef;     // ground-state pass: psi += y_{j+1} f_{j+1}
    T *psi;
};

template <typename T>
__global__ void __launch_bounds__(kPersistThreads)
lanczos_persistent_kernel(DevModel M, PersistArgs<T> A)
{
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    __shared__ double red[32];
    const int64_t dim = M.dim_up * M.dim_dn;
    const int64_t gtid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t gstride = (int64_t)gridDim.x * blockDim.x;
    const T tt = (T)M.t, UU = (T)M.U;

    double c_cur = A.S->c_cur, c_prev = A.S->c_prev, beta = A.S->beta, amax = A.S->amax;
    const double tau = A.S->tau;
    int stop = A.S->stop, jdone = A.S->j;

    for (int j = A.j0; j < A.j1 && !stop; ++j) {
        T *cur = (j & 1) ? A.vec1 : A.vec0;
        T *prev = (j & 1) ? A.vec0 : A.vec1;
        const T cc = (T)c_cur, bc = (T)(beta * c_prev);
        const T yc = A.psi ? (T)(A.ycoef[j] * c_cur) : T(0);
        // ---- lines 4-5 (+ eq. 13): q = H f_j - b_j f_{j-1} over f_{j-1}, a_j = q . f_j
        double acc = 0.0;
        for (int64_t J = gtid; J < dim; J += gstride) {
            const int64_t a = J / M.dim_dn, b = J - a * M.dim_dn;
            const T *xa = cur + a * M.dim_dn;
            T sum = T(0);
            const int nup = M.up_cnt[a];
            const uint32_t *ue = M.up_ent + a * M.w_up;
            for (int k = 0; k < nup; ++k) {                                   // Algorithm 2
                const uint32_t e = ue[k];
                sum += signed_by(e, cur[(int64_t)(e >> 1) * M.dim_dn + b]);
            }
            const int ndn = M.dn_cnt[b];
            for (int k = 0; k < ndn; ++k) {                                   // Algorithm 3
                const uint32_t e = M.dn_ent32[(int64_t)k * M.ld_dn + b];
                sum += signed_by(e, xa[e >> 1]);
            }
            const T xv = xa[b];
            const T h = tt * sum + UU * (T)__popc(M.st_up[a] & M.st_dn[b]) * xv;   // Algorithm 4
            const T q = cc * h - bc * prev[J];
            prev[J] = q;
            acc += (double)q * (double)(cc * xv);
            if (A.psi) A.psi[J] = fma(yc, xv, A.psi[J]);
        }
        double s = block_sum(acc, red);
        if (threadIdx.x == 0) A.part_a[blockIdx.x] = s;
        __threadfence();
        grid.sync();
        const double alpha = sum_partials(A.part_a, gridDim.x, red);
        __shared__ double bcast;
        if (threadIdx.x == 0) bcast = alpha;
        __syncthreads();
        const double a_j = bcast;
        // ---- lines 6-7: w = q - a_j f_j, b_{j+1} = |w|
        const T ac = (T)(a_j * c_cur);
        acc = 0.0;
        for (int64_t J = gtid; J < dim; J += gstride) {
            const T w = prev[J] - ac * cur[J];
            prev[J] = w;
            acc += (double)w * (double)w;
        }
        s = block_sum(acc, red);
        if (threadIdx.x == 0) A.part_b[blockIdx.x] = s;
        __threadfence();
        grid.sync();
        const double b2 = sum_partials(A.part_b, gridDim.x, red);
        __syncthreads();
        if (threadIdx.x == 0) bcast = b2;
        __syncthreads();
        const double bnew = sqrt(bcast);
        // ---- lines 8-11 (identical in every block)
        if (blockIdx.x == 0 && threadIdx.x == 0) { A.alpha_out[jdone] = a_j; A.beta_out[jdone] = bnew; }
        amax = fmax(amax, fabs(a_j));
        ++jdone;
        if (!isfinite(bnew) || !(bnew > tau * fmax(1.0, amax))) {
            stop = 1;
        } else {
            c_prev = c_cur;
            c_cur = 1.0 / bnew;
            beta = bnew;
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        A.S->c_cur = c_cur; A.S->c_prev = c_prev; A.S->beta = beta; A.S->amax = amax;
        A.S->j = jdone; A.S->stop = stop;
    }
}

}  // namespace hub
