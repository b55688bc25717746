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
// one operator application and ONE fused vector kernel (x += d; r -= Minv w; d = c1 d + c2 r).
#include "sem_internal.h"

namespace {

template <typename T, typename TM>
__global__ void __launch_bounds__(256) k_cheb_init(int64_t n, const T* __restrict__ b, const T* __restrict__ q,
                                                   const TM* __restrict__ Minv, T inv_theta, T* __restrict__ x,
                                                   T* __restrict__ r, T* __restrict__ d) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const T m = (T)Minv[l];
        const T rl = m * (q ? b[l] - q[l] : b[l]);      // q == nullptr: zero initial guess
        if (!q || m == T(0)) x[l] = T(0);               // zero guess, or a Dirichlet node (S14)
        r[l] = rl;
        d[l] = rl * inv_theta;
    }
}

template <typename T>
__global__ void __launch_bounds__(256) k_mask_x(int64_t n, const double* __restrict__ Minv, T* __restrict__ x) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x)
        if (Minv[l] == 0.0) x[l] = T(0);
}

template <typename T, typename TM>
__global__ void __launch_bounds__(256) k_cheb_step(int64_t n, const T* __restrict__ w, const TM* __restrict__ Minv,
                                                   T c1, T c2, T* __restrict__ x, T* __restrict__ r,
                                                   T* __restrict__ d) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const T dl = d[l];
        x[l] += dl;
        const T rl = r[l] - (T)Minv[l] * w[l];
        r[l] = rl;
        d[l] = c1 * dl + c2 * rl;
    }
}

template <typename T>
__global__ void __launch_bounds__(256) k_axpy1(int64_t n, const T* __restrict__ d, T* __restrict__ x) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x)
        x[l] += d[l];
}

template <typename T>
int run(sem_ctx* c, const T* b, T* x, int order, double lmin, double lmax, bool zero_guess) {
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
    if (zero_guess) {
        k_cheb_init<T, double><<<grid, 256, 0, st>>>(n, b, (const T*)nullptr, c->d_Minv, (T)(1.0 / theta), x, r, d);
    } else {
        k_mask_x<T><<<grid, 256, 0, st>>>(n, c->d_Minv, x);
        if ((rc = sem_launch_ax_gs(c, x, w, prec, c->lambda, nullptr, nullptr))) return rc;
        k_cheb_init<T, double><<<grid, 256, 0, st>>>(n, b, (const T*)w, c->d_Minv, (T)(1.0 / theta), x, r, d);
    }
    for (int k = 1; k < order; ++k) {
        if ((rc = sem_launch_ax_gs(c, d, w, prec, c->lambda, nullptr, nullptr))) return rc;
        const double rho1 = 1.0 / (2.0 * sigma - rho);
        k_cheb_step<T, double><<<grid, 256, 0, st>>>(n, w, c->d_Minv, (T)(rho1 * rho), (T)(2.0 * rho1 / delta), x, r, d);
        rho = rho1;
    }
    k_axpy1<T><<<grid, 256, 0, st>>>(n, d, x);
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

}  // namespace

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
    if (prec == SEM_F32 && c->gmode == SEM_G_STORED && (rc = sem_build_g32(c))) return rc;
    for (int q = 0; q < 3; ++q)
        if (!c->d_cheb[q]) SEM_CUDA_OK(c, cudaMalloc(&c->d_cheb[q], c->nL * sizeof(double)));
    if (prec == SEM_F64) return run<double>(c, (const double*)b, (double*)x, order, lmin, lmax, zero_guess != 0);
    return run<float>(c, (const float*)b, (float*)x, order, lmin, lmax, zero_guess != 0);
}
