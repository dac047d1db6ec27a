// Lanczos vector sweeps (Algorithm 1).  The paper is silent
// on how these are done; here each is one streaming sweep with a
// deterministic grid reduction, and the scalar bookkeeping of the iteration
// (lines 7-11) is done by the last block to arrive, so the host never
// synchronises inside the loop.
#pragma once
#include "kernels_common.cuh"

namespace hub {

constexpr int kVecThreads = 512;

template <typename T> struct Vec16;          // 16-byte vector of T
template <> struct Vec16<float>  { using type = float4;  static constexpr int n = 4; };
template <> struct Vec16<double> { using type = double2; static constexpr int n = 2; };

// ||v0||^2, then c_cur = 1/||v0|| (Algorithm 1 "Require: f_1 of norm 1": the
// caller's vector is normalised by scalar, its copy u_cur is left unscaled).
template <typename T>
__global__ void __launch_bounds__(kVecThreads)
lanczos_init_kernel(const T *__restrict__ u, int64_t dim, LanczosScalars *S, double *partials, double tau)
{
    __shared__ double red[32];
    __shared__ int flag;
    using V = typename Vec16<T>::type;
    constexpr int N = Vec16<T>::n;
    const int64_t nvec = dim / N;
    const int64_t per = (nvec + gridDim.x - 1) / gridDim.x;
    const int64_t lo = blockIdx.x * per, hi = min(nvec, lo + per);
    double acc = 0.0;
    for (int64_t i = lo + threadIdx.x; i < hi; i += blockDim.x) {
        V v = reinterpret_cast<const V *>(u)[i];
        const T *e = reinterpret_cast<const T *>(&v);
#pragma unroll
        for (int k = 0; k < N; ++k) acc += (double)e[k] * (double)e[k];
    }
    if (blockIdx.x == gridDim.x - 1)
        for (int64_t i = nvec * N + threadIdx.x; i < dim; i += blockDim.x) acc += (double)u[i] * (double)u[i];
    double s = block_sum(acc, red);
    if (publish_and_check_last(s, partials, blockIdx.x, gridDim.x, &S->ticket, &flag)) {
        double n2 = sum_partials(partials, gridDim.x, red);
        if (threadIdx.x == 0) {
            double nrm = sqrt(n2);
            bool ok = isfinite(nrm) && nrm > 0.0;
            S->c_cur = ok ? 1.0 / nrm : 0.0;
            S->c_prev = 0.0;
            S->beta = 0.0;       // line 1: b_1 <- 0
            S->alpha = 0.0;
            S->amax = 0.0;
            S->tau = tau;
            S->j = 0;
            S->stop = ok ? 0 : 1;
            S->ticket = 0;
        }
    }
}

// Lines 6-11: w <- w - a_j f_j (f_j = c_cur u_cur), b_{j+1} = ||w||; the last
// block records a_j, b_{j+1}, applies the breakdown rule (reading Q11) and
// rotates the scalars: f_{j+1} = w / b_{j+1} is carried as c_cur = 1/b_{j+1}.
template <typename T>
__global__ void __launch_bounds__(kVecThreads)
lanczos_axpy_norm_kernel(const T *__restrict__ u, T *__restrict__ w, int64_t dim, LanczosScalars *S,
                         double *partials, double *alpha_out, double *beta_out)
{
    __shared__ double red[32];
    __shared__ int flag;
    if (S->stop) return;
    using V = typename Vec16<T>::type;
    constexpr int N = Vec16<T>::n;
    const T ac = (T)(S->alpha * S->c_cur);
    const int64_t nvec = dim / N;
    const int64_t per = (nvec + gridDim.x - 1) / gridDim.x;
    const int64_t lo = blockIdx.x * per, hi = min(nvec, lo + per);
    double acc = 0.0;
    for (int64_t i = lo + threadIdx.x; i < hi; i += blockDim.x) {
        V uv = reinterpret_cast<const V *>(u)[i];
        V wv = reinterpret_cast<V *>(w)[i];
        const T *ue = reinterpret_cast<const T *>(&uv);
        T *we = reinterpret_cast<T *>(&wv);
#pragma unroll
        for (int k = 0; k < N; ++k) {
            we[k] = we[k] - ac * ue[k];
            acc += (double)we[k] * (double)we[k];
        }
        reinterpret_cast<V *>(w)[i] = wv;
    }
    if (blockIdx.x == gridDim.x - 1)
        for (int64_t i = nvec * N + threadIdx.x; i < dim; i += blockDim.x) {
            T q = w[i] - ac * u[i];
            w[i] = q;
            acc += (double)q * (double)q;
        }
    double s = block_sum(acc, red);
    if (publish_and_check_last(s, partials, blockIdx.x, gridDim.x, &S->ticket, &flag)) {
        double b2 = sum_partials(partials, gridDim.x, red);
        if (threadIdx.x == 0) {
            double beta = sqrt(b2), alpha = S->alpha;
            int j = S->j;
            alpha_out[j] = alpha;
            beta_out[j] = beta;
            double amax = fmax(S->amax, fabs(alpha));
            S->amax = amax;
            S->j = j + 1;
            if (!isfinite(beta) || !(beta > S->tau * fmax(1.0, amax))) {
                S->stop = 1;                      // lines 8-10
            } else {
                S->c_prev = S->c_cur;             // line 11, carried lazily
                S->c_cur = 1.0 / beta;
                S->beta = beta;
            }
            S->ticket = 0;
        }
    }
}

// ---- ground-state vector (second Lanczos pass, "the basis is not kept")
// psi += y_j f_j with f_j = c_cur * u (the scalars are those of the run in flight).
template <typename T>
__global__ void __launch_bounds__(kVecThreads)
psi_axpy_kernel(T *__restrict__ psi, const T *__restrict__ u, int64_t n, const double *__restrict__ ycoef,
                const LanczosScalars *S)
{
    if (S->stop) return;
    const T a = (T)(*ycoef * S->c_cur);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        psi[i] = fma(a, u[i], psi[i]);
}

// |x|^2 into S->beta (deterministic, as every other reduction here), then x *= 1 / sqrt(S->beta).
template <typename T>
__global__ void __launch_bounds__(kVecThreads)
vec_norm2_kernel(const T *__restrict__ x, int64_t n, LanczosScalars *S, double *partials)
{
    __shared__ double red[32];
    __shared__ int flag;
    double acc = 0.0;
    const int64_t per = (n + gridDim.x - 1) / gridDim.x;
    const int64_t lo = blockIdx.x * per, hi = min(n, lo + per);
    for (int64_t i = lo + threadIdx.x; i < hi; i += blockDim.x) acc += (double)x[i] * (double)x[i];
    const double s = block_sum(acc, red);
    if (publish_and_check_last(s, partials, blockIdx.x, gridDim.x, &S->ticket, &flag)) {
        const double tot = sum_partials(partials, gridDim.x, red);
        if (threadIdx.x == 0) { S->beta = tot; S->ticket = 0; }
    }
}

template <typename T>
__global__ void __launch_bounds__(kVecThreads)
vec_normalise_kernel(T *__restrict__ x, int64_t n, const LanczosScalars *S)
{
    const double n2 = S->beta;
    const T a = (T)((n2 > 0.0) ? rsqrt(n2) : 0.0);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) x[i] *= a;
}

// Complex propagation (lanczos_propagate_complex): A = sum_j Re(y_j) f_j and B = sum_j Im(y_j) f_j over the stacked
// vectors f_j = [g_j ; h_j] (real part ; imaginary part); (y f) = (Re y g - Im y h) + i (Re y h + Im y g).
template <typename T>
__global__ void __launch_bounds__(kVecThreads)
complex_mix_kernel(const T *__restrict__ A, const T *__restrict__ B, int64_t n, T *__restrict__ out_re, T *__restrict__ out_im)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        out_re[i] = A[i] - B[n + i];
        if (out_im) out_im[i] = A[n + i] + B[i];
    }
}

// ---- row-sharded Lanczos: the vector updates of Algorithm 1 on ONE rank's shard of n elements.  The
// scalars a_j, b_j come from the caller (all-reduced over the ranks); each kernel leaves its partial sum in
// partials[0..gridDim.x) and the fixed-order total in *result (device), which the caller all-reduces.
//   mode 0:  q = hf - b fprev   (lines 4 with eq. 13; written over fprev),  result = q . f      (line 5)
//   mode 1:  w = q  - a f       (line 6; in place),                         result = w . w      (line 7)
//   mode 2:  w = s w            (line 11)
template <typename T, int MODE>
__global__ void __launch_bounds__(kVecThreads)
shard_update_kernel(T *__restrict__ inout, const T *__restrict__ other, const T *__restrict__ f, int64_t n, double coef,
                    double *partials, unsigned *ticket, double *result)
{
    __shared__ double red[32];
    __shared__ int flag;
    const T cf = (T)coef;
    double acc = 0.0;
    const int64_t per = (n + gridDim.x - 1) / gridDim.x;
    const int64_t lo = blockIdx.x * per, hi = min(n, lo + per);
    for (int64_t i = lo + threadIdx.x; i < hi; i += blockDim.x) {
        if (MODE == 0) {
            const T q = other[i] - cf * inout[i];
            inout[i] = q;
            acc += (double)q * (double)f[i];
        } else if (MODE == 1) {
            const T w = inout[i] - cf * f[i];
            inout[i] = w;
            acc += (double)w * (double)w;
        } else {
            inout[i] = cf * inout[i];
        }
    }
    if (MODE == 2) return;
    const double s = block_sum(acc, red);
    if (publish_and_check_last(s, partials, blockIdx.x, gridDim.x, ticket, &flag)) {
        const double tot = sum_partials(partials, gridDim.x, red);
        if (threadIdx.x == 0) { *result = tot; *ticket = 0; }
    }
}

}  // namespace hub
