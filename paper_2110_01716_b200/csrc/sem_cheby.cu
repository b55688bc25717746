// sem_cheby.cu — NEXT-1: Chebyshev-accelerated point-Jacobi smoother of the p-multigrid
// preconditioner.  P:103 "Smoothers for pMG include Chebyshev-accelerated point-Jacobi"; "all steps of pMG in
// 32-bit arithmetic" (FP32 and FP64 are both provided).  The paper names the smoother only; the reading (S23)
// is the textbook Chebyshev semi-iteration on M^-1 A, M = diag(A) (the exact Jacobi diagonal O7), for caller-supplied
// eigenvalue bounds [lmin, lmax] of M^-1 A:
//   theta = (lmax+lmin)/2, delta = (lmax-lmin)/2, sigma = theta/delta, rho_0 = 1/sigma
//   r = M^-1 (b - A x);  d = r / theta
//   k = 1 .. order-1:  x += d;  r -= M^-1 A d;  rho_k = 1/(2 sigma - rho_{k-1});  d = rho_k rho_{k-1} d + (2 rho_k/delta) r
//   x += d
// A = M QQ^T (D^T G D + lambda B) M through sem_launch_ax_gs; every vector in local layout and continuous.  All the
// recurrence scalars depend on the bounds only, so they are computed on the host and nothing synchronises: per step
// one operator application and ONE fused vector kernel (x += d; r -= Minv w; d = c1 d + c2 r); the final x += d is
// folded into the last step, which then writes only x, and a zero initial guess is never read or pre-zeroed.
#include <math.h>
#include <stdlib.h>

#include <mutex>

#include "sem_internal.h"

namespace {

// r = Minv (b - q) (q == nullptr: zero initial guess); d = r / theta.  ONLY (order == 1): x <- x0 + d and nothing else
// is written.  Otherwise x is only masked here (non-zero guess) or not touched at all (zero guess: the first step
// writes it).
template <typename T, bool ONLY>
__global__ void __launch_bounds__(256) k_cheb_first(int64_t n, const T* __restrict__ b, const T* __restrict__ q,
                                                    const T* __restrict__ Minv, T inv_theta, T* __restrict__ x,
                                                    T* __restrict__ r, T* __restrict__ d) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const T m = Minv[l];
        const T rl = m * (q ? b[l] - q[l] : b[l]);
        const T dl = rl * inv_theta;
        if constexpr (ONLY) {
            x[l] = (q && m != T(0)) ? x[l] + dl : dl;     // Dirichlet node (m == 0): dl == 0
        } else {
            r[l] = rl;
            d[l] = dl;
        }
    }
}

template <typename T>
__global__ void __launch_bounds__(256) k_mask_x(int64_t n, const T* __restrict__ Minv, T* __restrict__ x) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x)
        if (Minv[l] == T(0)) x[l] = T(0);
}

// One step.  XZERO: x is (implicitly) zero before this step (zero guess, first step).  LAST: the final x += d is
// folded in and r, d are not written back:  x <- x + d + (c1 d + c2 (r - Minv w)).
template <typename T, bool XZERO, bool LAST>
__global__ void __launch_bounds__(256) k_cheb_step(int64_t n, const T* __restrict__ w, const T* __restrict__ Minv,
                                                   T c1, T c2, T* __restrict__ x, T* __restrict__ r,
                                                   T* __restrict__ d) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const T dl = d[l];
        const T rl = r[l] - Minv[l] * w[l];
        const T dn = c1 * dl + c2 * rl;
        const T x0 = XZERO ? T(0) : x[l];
        if constexpr (LAST) {
            x[l] = x0 + dl + dn;
        } else {
            x[l] = x0 + dl;
            r[l] = rl;
            d[l] = dn;
        }
    }
}

__global__ void __launch_bounds__(256) k_minv32(int64_t n, const double* __restrict__ a, float* __restrict__ o) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x)
        o[l] = (float)a[l];
}

template <typename T>
int run(sem_ctx* c, const T* b, T* x, int order, double lmin, double lmax, bool zero_guess) {
    cudaStream_t st = c->stream;
    const int64_t n = c->nL;
    const sem_prec prec = sizeof(T) == 8 ? SEM_F64 : SEM_F32;
    T* r = (T*)c->d_cheb[0];
    T* d = (T*)c->d_cheb[1];
    T* w = (T*)c->d_cheb[2];
    const T* Minv = sizeof(T) == 8 ? (const T*)c->d_Minv : (const T*)c->d_Minv32;
    const unsigned grid = (unsigned)c->num_sms * 8;
    const double theta = 0.5 * (lmax + lmin), delta = 0.5 * (lmax - lmin), sigma = theta / delta;
    double rho = 1.0 / sigma;
    int rc;
    const T* q = nullptr;
    if (!zero_guess) {
        k_mask_x<T><<<grid, 256, 0, st>>>(n, Minv, x);
        if ((rc = sem_launch_ax_gs(c, x, w, prec, c->lambda, nullptr, nullptr))) return rc;
        q = w;
    }
    if (order == 1) k_cheb_first<T, true><<<grid, 256, 0, st>>>(n, b, q, Minv, (T)(1.0 / theta), x, r, d);
    else k_cheb_first<T, false><<<grid, 256, 0, st>>>(n, b, q, Minv, (T)(1.0 / theta), x, r, d);
    for (int k = 1; k < order; ++k) {
        if ((rc = sem_launch_ax_gs(c, d, w, prec, c->lambda, nullptr, nullptr))) return rc;
        const double rho1 = 1.0 / (2.0 * sigma - rho);
        const T c1 = (T)(rho1 * rho), c2 = (T)(2.0 * rho1 / delta);
        const bool xzero = zero_guess && k == 1, last = k == order - 1;
        if (xzero && last) k_cheb_step<T, true, true><<<grid, 256, 0, st>>>(n, w, Minv, c1, c2, x, r, d);
        else if (xzero) k_cheb_step<T, true, false><<<grid, 256, 0, st>>>(n, w, Minv, c1, c2, x, r, d);
        else if (last) k_cheb_step<T, false, true><<<grid, 256, 0, st>>>(n, w, Minv, c1, c2, x, r, d);
        else k_cheb_step<T, false, false><<<grid, 256, 0, st>>>(n, w, Minv, c1, c2, x, r, d);
        rho = rho1;
    }
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

// ---- the same recurrence with the Schwarz operator S (sem_schwarz.cu) in place of diag^-1: r and w hold S-applied
// vectors, so the vector kernels carry no Minv ----
// r = b - q (q == nullptr: r = b)
template <typename T>
__global__ void __launch_bounds__(256) k_pc_resid(int64_t n, const T* __restrict__ b, const T* __restrict__ q,
                                                  T* __restrict__ r) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x)
        r[l] = q ? b[l] - q[l] : b[l];
}
// d = r / theta;  ONLY (order == 1): x <- x0 + d (x0 = 0 with a zero guess)
template <typename T, bool ONLY>
__global__ void __launch_bounds__(256) k_pc_first(int64_t n, const T* __restrict__ r, T inv_theta, bool xzero,
                                                  T* __restrict__ x, T* __restrict__ d) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const T dl = r[l] * inv_theta;
        if constexpr (ONLY) x[l] = xzero ? dl : x[l] + dl;
        else d[l] = dl;
    }
}
// x += d; r -= w (w = S A d); d = c1 d + c2 r; LAST folds the final x += d in
template <typename T, bool XZERO, bool LAST>
__global__ void __launch_bounds__(256) k_pc_step(int64_t n, const T* __restrict__ w, T c1, T c2, T* __restrict__ x,
                                                 T* __restrict__ r, T* __restrict__ d) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const T dl = d[l];
        const T rl = r[l] - w[l];
        const T dn = c1 * dl + c2 * rl;
        const T x0 = XZERO ? T(0) : x[l];
        if constexpr (LAST) x[l] = x0 + dl + dn;
        else { x[l] = x0 + dl; r[l] = rl; d[l] = dn; }
    }
}

template <typename T>
int run_schwarz(sem_ctx* c, const T* b, T* x, int order, double lmin, double lmax, bool zero_guess, int kind) {
    cudaStream_t st = c->stream;
    const int64_t n = c->nL;
    const sem_prec prec = sizeof(T) == 8 ? SEM_F64 : SEM_F32;
    T* r = (T*)c->d_cheb[0];
    T* d = (T*)c->d_cheb[1];
    T* w = (T*)c->d_cheb[2];
    const unsigned grid = (unsigned)c->num_sms * 8;
    const double theta = 0.5 * (lmax + lmin), delta = 0.5 * (lmax - lmin), sigma = theta / delta;
    double rho = 1.0 / sigma;
    int rc;
    // S is applied out of place (its restricted variant is then one fused kernel): t receives S(.)
    T* t = (T*)c->d_cheb4;
    if (!zero_guess) {
        if ((rc = sem_launch_ax_gs(c, x, w, prec, c->lambda, nullptr, nullptr))) return rc;      // x is masked on entry
        k_pc_resid<T><<<grid, 256, 0, st>>>(n, b, w, w);                                           // w = b - A x
        if ((rc = sem_launch_schwarz(c, w, r, prec, kind))) return rc;                             // r = S (b - A x)
    } else {
        if ((rc = sem_launch_schwarz(c, b, r, prec, kind))) return rc;                             // r = S b
    }
    if (order == 1) k_pc_first<T, true><<<grid, 256, 0, st>>>(n, r, (T)(1.0 / theta), zero_guess, x, d);
    else k_pc_first<T, false><<<grid, 256, 0, st>>>(n, r, (T)(1.0 / theta), zero_guess, x, d);
    for (int k = 1; k < order; ++k) {
        if ((rc = sem_launch_ax_gs(c, d, w, prec, c->lambda, nullptr, nullptr))) return rc;
        if ((rc = sem_launch_schwarz(c, w, t, prec, kind))) return rc;                           // t = S A d
        const double rho1 = 1.0 / (2.0 * sigma - rho);
        const T c1 = (T)(rho1 * rho), c2 = (T)(2.0 * rho1 / delta);
        const bool xzero = zero_guess && k == 1, last = k == order - 1;
        if (xzero && last) k_pc_step<T, true, true><<<grid, 256, 0, st>>>(n, t, c1, c2, x, r, d);
        else if (xzero) k_pc_step<T, true, false><<<grid, 256, 0, st>>>(n, t, c1, c2, x, r, d);
        else if (last) k_pc_step<T, false, true><<<grid, 256, 0, st>>>(n, t, c1, c2, x, r, d);
        else k_pc_step<T, false, false><<<grid, 256, 0, st>>>(n, t, c1, c2, x, r, d);
        rho = rho1;
    }
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

// power iteration helpers: v = Minv * w, s[0] += wt v v   /   v *= scale
__global__ void __launch_bounds__(256) k_pow_apply(int64_t n, const double* __restrict__ w, const double* __restrict__ Minv,
                                                   const double* __restrict__ wt, double* __restrict__ v,
                                                   double* __restrict__ s) {
    double acc = 0.0;
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const double vl = Minv ? Minv[l] * w[l] : w[l];      // Minv == nullptr: w already holds S A v
        v[l] = vl;
        acc += wt[l] * vl * vl;
    }
    __shared__ double red[32];
    for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        acc = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.0;
        for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (threadIdx.x == 0) atomicAdd(s, acc);
    }
}
__global__ void __launch_bounds__(256) k_pow_scale(int64_t n, double a, double* __restrict__ v) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) v[l] *= a;
}
// a rough, continuous, masked start vector: a hash of the unique node index (an under-estimate of lmax makes the
// smoother amplify the modes above it, so the start must not be smooth)
__global__ void __launch_bounds__(256) k_pow_start(int64_t n, const int32_t* __restrict__ l2u, const double* __restrict__ wt,
                                                   double* __restrict__ v) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        uint32_t h = (uint32_t)l2u[l] * 2654435761u;
        h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
        v[l] = wt[l] != 0.0 ? (double)(h & 0xffffu) / 32768.0 - 1.0 : 0.0;
    }
}

}  // namespace

// Largest eigenvalue of diag^-1 A by `iters` power iterations (setup helper for sem_cheby / sem_pmg_create, S23):
// returns the last Rayleigh-type estimate ||diag^-1 A v|| / ||v|| (a lower bound that converges from below; callers
// multiply by a safety factor, usually 1.1).  FP64; synchronises once per iteration.
extern "C" int sem_lambda_max(sem_ctx* c, int iters, double* lam_out) {
    if (!c || !lam_out) return SEM_EINVAL;
    c->err.clear();
    if (iters < 1) return sem_fail(c, SEM_EINVAL, "sem_lambda_max: iters < 1");
    if (!c->geom_done) return sem_fail(c, SEM_ESTATE, "sem_lambda_max before sem_geom");
    int rc;
    if (!c->d_Minv || c->lambda_of_diag != c->lambda) {
        if ((rc = sem_build_diag(c))) return rc;
    }
    for (int q = 0; q < 3; ++q)
        if (!c->d_cheb[q]) SEM_CUDA_OK(c, cudaMalloc(&c->d_cheb[q], c->nL * sizeof(double)));
    double *v = (double*)c->d_cheb[0], *w = (double*)c->d_cheb[1], *s = (double*)c->d_cheb[2];
    cudaStream_t st = c->stream;
    const unsigned grid = (unsigned)c->num_sms * 8;
    k_pow_start<<<grid, 256, 0, st>>>(c->nL, c->d_l2u, c->d_wt, v);
    double lam = 0.0;                                     // iteration 0 only normalises the start vector
    for (int it = 0; it <= iters; ++it) {
        SEM_CUDA_OK(c, cudaMemsetAsync(s, 0, sizeof(double), st));
        if ((rc = sem_launch_ax_gs(c, v, w, SEM_F64, c->lambda, nullptr, nullptr))) return rc;
        k_pow_apply<<<grid, 256, 0, st>>>(c->nL, w, c->d_Minv, c->d_wt, v, s);
        double h = 0.0;
        SEM_CUDA_OK(c, cudaMemcpyAsync(&h, s, sizeof(double), cudaMemcpyDeviceToHost, st));
        SEM_CUDA_OK(c, cudaStreamSynchronize(st));
        const double wnorm = sqrt(h);
        if (!(wnorm > 0.0)) return sem_fail(c, SEM_EINVAL, "sem_lambda_max: operator annihilates the start vector");
        if (it > 0) lam = wnorm;                          // v had unit norm
        k_pow_scale<<<grid, 256, 0, st>>>(c->nL, 1.0 / wnorm, v);
    }
    SEM_CUDA_OK(c, cudaGetLastError());
    *lam_out = lam;
    return SEM_OK;
}

extern "C" int sem_cheby(sem_ctx* c, const void* b, void* x, int order, double lmin, double lmax, int zero_guess,
                         sem_prec prec) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (!b || !x || b == x) return sem_fail(c, SEM_EINVAL, "sem_cheby: NULL or aliased vectors");
    if (prec != SEM_F64 && prec != SEM_F32) return sem_fail(c, SEM_EINVAL, "sem_cheby: bad sem_prec");
    if (order < 1 || !(lmin > 0.0) || !(lmax > lmin))
        return sem_fail(c, SEM_EINVAL, "sem_cheby: need order >= 1 and 0 < lmin < lmax");
    if (((uintptr_t)x % 16) || ((uintptr_t)b % (prec == SEM_F64 ? 8 : 4)))
        return sem_fail(c, SEM_EINVAL, "sem_cheby: x must be 16-byte aligned");
    if (!c->geom_done) return sem_fail(c, SEM_ESTATE, "sem_cheby before sem_geom");
    if (c->lambda != 0.0 && !c->with_mass) return sem_fail(c, SEM_ESTATE, "lambda != 0 needs with_mass");
    int rc;
    if (!c->d_Minv || c->lambda_of_diag != c->lambda) {
        if ((rc = sem_build_diag(c))) return rc;
    }
    if (prec == SEM_F32 && (rc = sem_build_g32(c))) return rc;
    for (int q = 0; q < 3; ++q)
        if (!c->d_cheb[q]) SEM_CUDA_OK(c, cudaMalloc(&c->d_cheb[q], c->nL * sizeof(double)));
    if (prec == SEM_F32 && (!c->d_Minv32 || c->lambda_of_minv32 != c->lambda)) {       // S16: rounded once from double
        if (!c->d_Minv32) SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_Minv32, c->nL * sizeof(float)));
        k_minv32<<<(unsigned)c->num_sms * 8, 256, 0, c->stream>>>(c->nL, c->d_Minv, c->d_Minv32);
        c->lambda_of_minv32 = c->lambda;
    }
    // N = 1 (the coarsest multigrid level): the operator is assembled once and a whole step is one kernel (sem_coarse.cu).
    // The assembly runs operator applications and synchronises, so it happens on an eager call, never inside a capture.
    if (c->p == 2 && c->gmode == SEM_G_STORED) {
        const char* env = getenv("SEM_COARSE");
        if (!(env && env[0] == '0')) {
            cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
            if (c->stream != cudaStreamLegacy && c->stream != nullptr) cudaStreamIsCapturing(c->stream, &cs);
            const bool have = c->coarse != nullptr && sem_coarse_is_current(c);
            if (have || cs == cudaStreamCaptureStatusNone) {
                if (!have && (rc = sem_coarse_build(c))) return rc;
                return sem_coarse_cheby(c, b, x, order, lmin, lmax, zero_guess != 0, prec);
            }
        }
    }
    if (prec == SEM_F64) return run<double>(c, (const double*)b, (double*)x, order, lmin, lmax, zero_guess != 0);
    return run<float>(c, (const float*)b, (float*)x, order, lmin, lmax, zero_guess != 0);
}


// Chebyshev-accelerated Schwarz: see include/sem.h.
extern "C" int sem_cheby_schwarz(sem_ctx* c, const void* b, void* x, int order, double lmin, double lmax, int zero_guess,
                                 sem_prec prec, sem_schwarz_kind kind) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (!b || !x || b == x) return sem_fail(c, SEM_EINVAL, "sem_cheby_schwarz: NULL or aliased vectors");
    if (prec != SEM_F64 && prec != SEM_F32) return sem_fail(c, SEM_EINVAL, "sem_cheby_schwarz: bad sem_prec");
    if (kind != SEM_SCHWARZ_ASM && kind != SEM_SCHWARZ_RAS) return sem_fail(c, SEM_EINVAL, "sem_cheby_schwarz: bad kind");
    if (order < 1 || !(lmin > 0.0) || !(lmax > lmin))
        return sem_fail(c, SEM_EINVAL, "sem_cheby_schwarz: need order >= 1 and 0 < lmin < lmax");
    if (((uintptr_t)x % 16) || ((uintptr_t)b % (prec == SEM_F64 ? 8 : 4)))
        return sem_fail(c, SEM_EINVAL, "sem_cheby_schwarz: x must be 16-byte aligned");
    if (!c->sw) return sem_fail(c, SEM_ESTATE, "sem_cheby_schwarz before sem_schwarz_setup");
    if (c->lambda != 0.0 && !c->with_mass) return sem_fail(c, SEM_ESTATE, "lambda != 0 needs with_mass");
    int rc;
    if (prec == SEM_F32 && (rc = sem_build_g32(c))) return rc;
    for (int q = 0; q < 3; ++q)
        if (!c->d_cheb[q]) SEM_CUDA_OK(c, cudaMalloc(&c->d_cheb[q], c->nL * sizeof(double)));
    if (!c->d_cheb4) SEM_CUDA_OK(c, cudaMalloc(&c->d_cheb4, c->nL * sizeof(double)));
    if (prec == SEM_F64)
        return run_schwarz<double>(c, (const double*)b, (double*)x, order, lmin, lmax, zero_guess != 0, (int)kind);
    return run_schwarz<float>(c, (const float*)b, (float*)x, order, lmin, lmax, zero_guess != 0, (int)kind);
}

extern "C" int sem_lambda_max_schwarz(sem_ctx* c, sem_schwarz_kind kind, int iters, double* lam_out) {
    if (!c || !lam_out) return SEM_EINVAL;
    c->err.clear();
    if (iters < 1) return sem_fail(c, SEM_EINVAL, "sem_lambda_max_schwarz: iters < 1");
    if (kind != SEM_SCHWARZ_ASM && kind != SEM_SCHWARZ_RAS) return sem_fail(c, SEM_EINVAL, "bad sem_schwarz_kind");
    if (!c->sw) return sem_fail(c, SEM_ESTATE, "sem_lambda_max_schwarz before sem_schwarz_setup");
    int rc;
    if (!c->d_Minv || c->lambda_of_diag != c->lambda) {
        if ((rc = sem_build_diag(c))) return rc;              // the dot weights wt
    }
    for (int q = 0; q < 3; ++q)
        if (!c->d_cheb[q]) SEM_CUDA_OK(c, cudaMalloc(&c->d_cheb[q], c->nL * sizeof(double)));
    double *v = (double*)c->d_cheb[0], *w = (double*)c->d_cheb[1], *s = (double*)c->d_cheb[2];
    cudaStream_t st = c->stream;
    const unsigned grid = (unsigned)c->num_sms * 8;
    k_pow_start<<<grid, 256, 0, st>>>(c->nL, c->d_l2u, c->d_wt, v);
    double lam = 0.0;
    for (int it = 0; it <= iters; ++it) {
        SEM_CUDA_OK(c, cudaMemsetAsync(s, 0, sizeof(double), st));
        if ((rc = sem_launch_ax_gs(c, v, w, SEM_F64, c->lambda, nullptr, nullptr))) return rc;
        if ((rc = sem_launch_schwarz(c, w, w, SEM_F64, (int)kind))) return rc;
        k_pow_apply<<<grid, 256, 0, st>>>(c->nL, w, nullptr, c->d_wt, v, s);
        double h = 0.0;
        SEM_CUDA_OK(c, cudaMemcpyAsync(&h, s, sizeof(double), cudaMemcpyDeviceToHost, st));
        SEM_CUDA_OK(c, cudaStreamSynchronize(st));
        const double wnorm = sqrt(h);
        if (!(wnorm > 0.0)) return sem_fail(c, SEM_EINVAL, "sem_lambda_max_schwarz: operator annihilates the start vector");
        if (it > 0) lam = wnorm;
        k_pow_scale<<<grid, 256, 0, st>>>(c->nL, 1.0 / wnorm, v);
    }
    SEM_CUDA_OK(c, cudaGetLastError());
    *lam_out = lam;
    return SEM_OK;
}


// ---------------------------------------------------------------------------------------------------------------
// sem_cheby_noalloc: the Chebyshev-Jacobi smoother (FP64) for callers that cannot allocate device memory -- code under
// CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  sem_cheby allocates its three work
// vectors (and, if needed, the Jacobi diagonal) on first use; this entry point allocates NOTHING: r, d, w live in the
// file-scope array below (3 x SEM_NOALLOC_MAX_NODES doubles = 12 MB, part of the library image: every GPU that loads
// the library holds it until the process exits), and the Jacobi diagonal must already be current.
// The array's name is a device symbol: in host code it is only a stand-in, so its device address is resolved once per
// device with cudaGetSymbolAddress (that device current) and that pointer is what the kernels get.
// All calls (all contexts on a device) share the array; it keeps the last call's contents, and every value a call reads
// from it was written earlier by the same call (k_cheb_first writes all of r and d, the operator all of w), so nothing
// has to be cleared.  Two calls that overlap on the GPU (different streams) race on it.
// ---------------------------------------------------------------------------------------------------------------
static __device__ __align__(256) double sem_noalloc_scratch[3 * (size_t)SEM_NOALLOC_MAX_NODES];

namespace {

std::mutex noalloc_mu;
double* noalloc_ptr[SEM_MAX_DEVICES] = {};      // device address of sem_noalloc_scratch, per device

// set-up, once per device: the context's device must be the current one
int noalloc_resolve(sem_ctx* c, double** out) {
    if (c->device < 0 || c->device >= SEM_MAX_DEVICES) return sem_fail(c, SEM_EINVAL, "sem_cheby_noalloc: device index out of range");
    int cur = -1;
    SEM_CUDA_OK(c, cudaGetDevice(&cur));
    if (cur != c->device) return sem_fail(c, SEM_ESTATE, "sem_cheby_noalloc: the context's device %d is not current (%d)", c->device, cur);
    std::lock_guard<std::mutex> lk(noalloc_mu);
    if (!noalloc_ptr[cur]) {
        double* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, sem_noalloc_scratch);
        if (e != cudaSuccess || !p) return sem_fail(c, SEM_ECUDA, "sem_cheby_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
        noalloc_ptr[cur] = p;
    }
    *out = noalloc_ptr[cur];
    return SEM_OK;
}

}  // namespace

extern "C" int sem_cheby_noalloc(sem_ctx* c, const double* b, double* x, int order, double lmin, double lmax,
                                 int zero_guess) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (!b || !x || b == x) return sem_fail(c, SEM_EINVAL, "sem_cheby_noalloc: NULL or aliased vectors");
    if (order < 1 || !(lmin > 0.0) || !(lmax > lmin))
        return sem_fail(c, SEM_EINVAL, "sem_cheby_noalloc: need order >= 1 and 0 < lmin < lmax");
    if (((uintptr_t)x % 16) || ((uintptr_t)b % 8)) return sem_fail(c, SEM_EINVAL, "sem_cheby_noalloc: x must be 16-byte aligned");
    if (c->nL > (int64_t)SEM_NOALLOC_MAX_NODES)
        return sem_fail(c, SEM_EINVAL, "sem_cheby_noalloc: %lld local nodes exceed SEM_NOALLOC_MAX_NODES = %d (use sem_cheby)",
                        (long long)c->nL, (int)SEM_NOALLOC_MAX_NODES);
    if (!c->geom_done) return sem_fail(c, SEM_ESTATE, "sem_cheby_noalloc before sem_geom");
    if (c->gmode != SEM_G_STORED) return sem_fail(c, SEM_ESTATE, "sem_cheby_noalloc needs stored geometric factors");
    if (c->lambda != 0.0 && !c->with_mass) return sem_fail(c, SEM_ESTATE, "lambda != 0 needs with_mass");
    if (!c->d_Minv || c->lambda_of_diag != c->lambda)
        return sem_fail(c, SEM_ESTATE, "sem_cheby_noalloc: the Jacobi diagonal is not built for this lambda "
                                       "(call sem_get_diag, sem_cheby or sem_pcg once before)");
    double* s = nullptr;
    int rc = noalloc_resolve(c, &s);
    if (rc) return rc;
    cudaStream_t st = c->stream;
    const int64_t n = c->nL;
    double *r = s, *d = s + SEM_NOALLOC_MAX_NODES, *w = s + 2 * (size_t)SEM_NOALLOC_MAX_NODES;
    const double* Minv = c->d_Minv;
    const unsigned grid = (unsigned)c->num_sms * 8;
    const double theta = 0.5 * (lmax + lmin), delta = 0.5 * (lmax - lmin), sigma = theta / delta;
    double rho = 1.0 / sigma;
    const double* q = nullptr;
    if (!zero_guess) {
        k_mask_x<double><<<grid, 256, 0, st>>>(n, Minv, x);
        if ((rc = sem_launch_ax_gs(c, x, w, SEM_F64, c->lambda, nullptr, nullptr))) return rc;
        q = w;
    }
    if (order == 1) k_cheb_first<double, true><<<grid, 256, 0, st>>>(n, b, q, Minv, 1.0 / theta, x, r, d);
    else k_cheb_first<double, false><<<grid, 256, 0, st>>>(n, b, q, Minv, 1.0 / theta, x, r, d);
    for (int k = 1; k < order; ++k) {
        if ((rc = sem_launch_ax_gs(c, d, w, SEM_F64, c->lambda, nullptr, nullptr))) return rc;
        const double rho1 = 1.0 / (2.0 * sigma - rho);
        const double c1 = rho1 * rho, c2 = 2.0 * rho1 / delta;
        const bool xzero = zero_guess && k == 1, last = k == order - 1;
        if (xzero && last) k_cheb_step<double, true, true><<<grid, 256, 0, st>>>(n, w, Minv, c1, c2, x, r, d);
        else if (xzero) k_cheb_step<double, true, false><<<grid, 256, 0, st>>>(n, w, Minv, c1, c2, x, r, d);
        else if (last) k_cheb_step<double, false, true><<<grid, 256, 0, st>>>(n, w, Minv, c1, c2, x, r, d);
        else k_cheb_step<double, false, false><<<grid, 256, 0, st>>>(n, w, Minv, c1, c2, x, r, d);
        rho = rho1;
    }
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}
