// Row sweep for sectors whose V row does not fit one SM's shared memory (C5 in
// fp64: 48 620 x 8 B = 380 KB; SURVEY.md hard part H3): a thread-block CLUSTER of
// NC CTAs holds R rows in distributed shared memory, each CTA one contiguous part
// of the contracted index, interleaved [j][R] as in variant GATHER.  A gather
// whose source lies in another part is a DSMEM load (ld.shared::cluster through
// the mapped generic address); on a ring only the hops over the highest sites
// change parts.  Same arithmetic as the row half of variant TWOSWEEP (Algorithm 3
// + Algorithm 4; eq. 13 in the Lanczos form), row-major in and
// out; hop entries in the batch-interleaved, bank-aware layout of variant GATHER
// (gather_tables.h).
#pragma once
#include <cooperative_groups.h>

#include "kernels_gather.cuh"

namespace hub {

constexpr int kClusterThreads = 1024;

template <typename T>
struct ClusterRowArgs {
    SpinDev in;              // down-spin table (layout for R rows, zero_base = dim_dn rounded up to R)
    const uint32_t *st_up;
    int64_t dim_up, dim_dn;
    int part;                // contracted indices per CTA (multiple of 32); the last rank holds the rest
    double t, U;
    const T *x;
    T *y;
    LanczosScalars *S;       // null: y = (t H_dn + D) x ; else y = c (...) - b c_prev y
};

template <typename T, typename E, int R, int NC>
__global__ void __launch_bounds__(kClusterThreads, 1)
row_cluster_kernel(ClusterRowArgs<T> A)
{
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using PR = Pack<T, R>;
    using EB = typename BatchOf<E>::type;
    PR *Xs = reinterpret_cast<PR *>(smem_raw);            // [my_n + kZero]
    constexpr int kZero = 128 / (int)sizeof(PR);          // zero slots, one per bank group (padding entries)

    const int rank = (int)cluster.block_rank();
    const int dd = (int)A.dim_dn;
    const int part = A.part;
    const int my0 = rank * part;                           // first contracted index this CTA holds
    const int my_n = max(0, min(dd, my0 + part) - my0);
    const int my_w = (my_n + 31) & ~31;
    const int zero_base = (dd + R - 1) / R * R;            // padding entries are zero_base + z
    const PR *base[NC];                                    // every CTA's part, as generic (DSMEM) addresses
#pragma unroll
    for (int r = 0; r < NC; ++r) base[r] = cluster.map_shared_rank(Xs, (unsigned)r);
    const E *__restrict__ ent = ent_ptr<E>(A.in);
    const int64_t ld = A.in.ld;
    const T tt = (T)A.t, UU = (T)A.U;
    T c = T(1), bcp = T(0);
    const bool stop = A.S && A.S->stop;                    // the same in every CTA of the cluster (cluster.sync below)
    if (A.S && !stop) { c = (T)A.S->c_cur; bcp = (T)(A.S->beta * A.S->c_prev); }
    if (threadIdx.x < kZero) {
        PR z;
#pragma unroll
        for (int r = 0; r < R; ++r) z.v[r] = T(0);
        Xs[my_n + threadIdx.x] = z;
    }
    const int64_t n_clusters = gridDim.x / NC, cid = blockIdx.x / NC;
    const int64_t n_tiles = (A.dim_up + R - 1) / R;

    for (int64_t tile = cid; tile < n_tiles && !stop; tile += n_clusters) {
        const int64_t a0 = tile * R;
        cluster.sync();                                    // every part is free (previous tile's gathers done)
        for (int j = threadIdx.x; j < my_n; j += kClusterThreads) {
            PR v;
#pragma unroll
            for (int r = 0; r < R; ++r) v.v[r] = (a0 + r < A.dim_up) ? A.x[(a0 + r) * dd + my0 + j] : T(0);
            Xs[j] = v;
        }
        cluster.sync();                                    // every part is staged
        uint32_t su[R];
#pragma unroll
        for (int r = 0; r < R; ++r) su[r] = (a0 + r < A.dim_up) ? A.st_up[a0 + r] : 0u;
        EB pk = load_batch(reinterpret_cast<const EB *>(ent) + my0 + min((int)threadIdx.x, max(my_w - 1, 0)));
        for (int il = threadIdx.x; il < my_w; il += kClusterThreads) {
            const int i = my0 + il;
            const bool valid = il < my_n;
            const int n = (int)A.in.wslots[i >> 5];        // slots every lane of this warp walks (my0 is a multiple of 32)
            const int nb = (n + kGatherBatch - 1) / kGatherBatch;
            const uint32_t sd = valid ? A.in.st[i] : 0u;
            T yold[R];
#pragma unroll
            for (int r = 0; r < R; ++r) yold[r] = (A.S && valid && a0 + r < A.dim_up) ? A.y[(a0 + r) * dd + i] : T(0);
            T acc[R];
#pragma unroll
            for (int r = 0; r < R; ++r) acc[r] = T(0);
            const EB *ep = reinterpret_cast<const EB *>(ent) + i;
            for (int b = 0; b < nb; ++b) {
                const EB *np = (b + 1 < nb) ? ep + ld
                                            : reinterpret_cast<const EB *>(ent) + my0 + min(il + kClusterThreads, my_w - 1);
                ep = np;
                const EB nxt = load_batch(np);
#pragma unroll
                for (int j = 0; j < kGatherBatch; ++j) {
                    int col;
                    T s;
                    if constexpr (sizeof(E) == 2) {      // packed 16-bit device entries (kernels_gather.cuh)
                        col = (int)packed_pos(pk, j);
                        s = packed_sign<T>(pk, j);
                    } else {
                        col = (int)(pk.v[j] >> 1);
                        s = sign_one<T>(pk.v[j]);
                    }
                    // one branch-free generic load: the owner's part (this CTA's own or another's through
                    // distributed shared memory), or a local zero slot for a padding entry
                    int owner = 0;
#pragma unroll
                    for (int r = 1; r < NC; ++r) owner += (col >= r * part) ? 1 : 0;
                    const PR *ob = base[0];
#pragma unroll
                    for (int r = 1; r < NC; ++r) ob = (owner == r) ? base[r] : ob;
                    const PR *src = ob + (col - owner * part);
                    src = (col >= dd) ? Xs + my_n + (col - zero_base) : src;
                    const PR v = *src;
#pragma unroll
                    for (int r = 0; r < R; ++r) acc[r] = fma(s, v.v[r], acc[r]);
                }
                pk = nxt;
            }
            if (valid) {
                const PR xv = Xs[il];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    if (a0 + r < A.dim_up) {
                        const T h = tt * acc[r] + UU * (T)__popc(su[r] & sd) * xv.v[r];      // Algorithm 4
                        A.y[(a0 + r) * dd + i] = A.S ? c * h - bcp * yold[r] : h;
                    }
                }
            }
        }
    }
    cluster.sync();                                        // no CTA exits while a peer may still read its part
}

}  // namespace hub
