// sem_proj.cu — NEXT-3: projection onto previous solutions.  P:111: "For any n x L subspace of R^n
// with A-orthonormal basis P_L = [p_1 ... p_L], the best-fit approximation to the solution of A p^m = b^m is
// pbar = P_L P_L^T b^m, which can be computed with a single allreduce of length L (<~ 30).  The residual for the reduced
// problem A dp = b^m - A pbar has a significantly smaller norm ... We augment the space P_{L+1} = [P_L dp] after
// orthonormalizing dp against P_L with one round of classical Gram-Schmidt ... L_max = 30 before restarting".
// Reading S27: A p_i is stored beside p_i (reduced right-hand side = b - sum alpha_i A p_i, no extra
// operator application); the A-norm of the orthogonalised direction comes from the same reduction; restart = empty the
// space; a direction with orthogonalised A-norm^2 <= 1e-12 of its own is dropped.
// These are the paper's tall-skinny, pure-bandwidth kernels: one pass over L (+1) vectors for the L dot products (the
// "single allreduce"), one pass over 2L vectors for the two updates.  All coefficients stay on the device.
#include <new>

#include "sem_internal.h"

struct sem_proj {
    sem_ctx* c = nullptr;
    int Lmax = 0, L = 0;
    double* P = nullptr;       // [Lmax][nL]
    double* AP = nullptr;      // [Lmax][nL]
    double* w = nullptr;       // [nL]   A dx
    double* coef = nullptr;    // [Lmax + 2] device coefficients: alpha / beta, then gamma
    int* flag = nullptr;       // device: 1 = last update accepted
};

namespace {

constexpr int CH = 8;          // basis vectors per pass of the multi-dot

// out[i] += sum_l wt_l B_i[l] v[l] for i = 0 .. cnt-1 (B_i = base + i*n), and out[cnt] += sum wt v2 v if v2
__global__ void __launch_bounds__(256) k_multidot(int64_t n, int cnt, const double* __restrict__ base,
                                                  const double* __restrict__ v, const double* __restrict__ v2,
                                                  const double* __restrict__ wt, double* __restrict__ out) {
    double acc[CH + 1];
#pragma unroll
    for (int i = 0; i <= CH; ++i) acc[i] = 0.0;
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const double wv = wt[l] * v[l];
#pragma unroll
        for (int i = 0; i < CH; ++i)
            if (i < cnt) acc[i] += base[(int64_t)i * n + l] * wv;
        if (v2) acc[CH] += v2[l] * wv;
    }
    __shared__ double red[8][CH + 1];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
    for (int i = 0; i <= CH; ++i) {
        double a = acc[i];
        for (int o = 16; o; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
        if (lane == 0) red[warp][i] = a;
    }
    __syncthreads();
    if (threadIdx.x <= CH) {
        double a = 0.0;
        for (int q = 0; q < 8; ++q) a += red[q][threadIdx.x];
        if (threadIdx.x < cnt) atomicAdd(out + threadIdx.x, a);
        else if (threadIdx.x == CH && v2) atomicAdd(out + cnt, a);
    }
}

// xbar = sum alpha_i P_i;  bred = b - sum alpha_i AP_i
__global__ void __launch_bounds__(256) k_guess(int64_t n, int L, const double* __restrict__ P, const double* __restrict__ AP,
                                               const double* __restrict__ alpha, const double* __restrict__ b,
                                               double* __restrict__ xbar, double* __restrict__ bred) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        double x = 0.0, r = b[l];
        for (int i = 0; i < L; ++i) {
            const double a = alpha[i];
            x += a * P[(int64_t)i * n + l];
            r -= a * AP[(int64_t)i * n + l];
        }
        xbar[l] = x;
        bred[l] = r;
    }
}

// P_L = (dx - sum beta_i P_i) s,  AP_L = (w - sum beta_i AP_i) s,  s = 1/sqrt(gamma - sum beta_i^2); dropped (flag = 0)
// if gamma <= 0 or the orthogonalised A-norm^2 is <= 1e-12 gamma
__global__ void __launch_bounds__(256) k_append(int64_t n, int L, const double* __restrict__ P, const double* __restrict__ AP,
                                                const double* __restrict__ coef, const double* __restrict__ dx,
                                                const double* __restrict__ w, double* __restrict__ Pn,
                                                double* __restrict__ APn, int* __restrict__ flag) {
    double nrm2 = coef[L];
    const double gamma = nrm2;
    for (int i = 0; i < L; ++i) nrm2 -= coef[i] * coef[i];
    const bool ok = gamma > 0.0 && nrm2 > 1e-12 * gamma;
    if (blockIdx.x == 0 && threadIdx.x == 0) *flag = ok ? 1 : 0;
    if (!ok) return;
    const double s = 1.0 / sqrt(nrm2);
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        double x = dx[l], y = w[l];
        for (int i = 0; i < L; ++i) {
            const double bta = coef[i];
            x -= bta * P[(int64_t)i * n + l];
            y -= bta * AP[(int64_t)i * n + l];
        }
        Pn[l] = x * s;
        APn[l] = y * s;
    }
}

int multidot(sem_proj* pj, const double* base, int cnt, const double* v, const double* v2) {
    sem_ctx* c = pj->c;
    SEM_CUDA_OK(c, cudaMemsetAsync(pj->coef, 0, (pj->Lmax + 2) * sizeof(double), c->stream));
    const unsigned grid = (unsigned)c->num_sms * 8;
    for (int i0 = 0; i0 < cnt || (i0 == 0 && v2); i0 += CH) {
        const int m = cnt - i0 < CH ? cnt - i0 : CH;
        const bool last = i0 + CH >= cnt;
        k_multidot<<<grid, 256, 0, c->stream>>>(c->nL, m, base + (int64_t)i0 * c->nL, v, last ? v2 : nullptr, c->d_wt,
                                                pj->coef + i0);
        if (cnt == 0) break;
    }
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

}  // namespace

extern "C" int sem_proj_create(sem_proj** out, sem_ctx* c, int Lmax) {
    if (!out) return SEM_EINVAL;
    *out = nullptr;
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (Lmax < 1 || Lmax > 64) return sem_fail(c, SEM_EINVAL, "sem_proj_create: need 1 <= Lmax <= 64");
    if (!c->geom_done) return sem_fail(c, SEM_ESTATE, "sem_proj_create before sem_geom");
    int rc;
    if (!c->d_wt || c->lambda_of_diag != c->lambda) {
        if ((rc = sem_build_diag(c))) return rc;          // wt: the unique-node dot weights
    }
    sem_proj* pj = new (std::nothrow) sem_proj();
    if (!pj) return SEM_ENOMEM;
    pj->c = c;
    pj->Lmax = Lmax;
    cudaError_t e = cudaMalloc((void**)&pj->P, (size_t)Lmax * c->nL * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&pj->AP, (size_t)Lmax * c->nL * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&pj->w, c->nL * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&pj->coef, (Lmax + 2) * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&pj->flag, sizeof(int));
    if (e != cudaSuccess) {
        sem_fail(c, SEM_ENOMEM, "sem_proj_create: %s", cudaGetErrorString(e));
        sem_proj_destroy(pj);
        return SEM_ENOMEM;
    }
    *out = pj;
    return SEM_OK;
}

extern "C" int sem_proj_guess(sem_proj* pj, const double* b, double* xbar, double* b_reduced) {
    if (!pj) return SEM_EINVAL;
    sem_ctx* c = pj->c;
    c->err.clear();
    if (!b || !xbar || !b_reduced || xbar == b_reduced) return sem_fail(c, SEM_EINVAL, "sem_proj_guess: NULL or aliased vectors");
    int rc;
    if ((rc = multidot(pj, pj->P, pj->L, b, nullptr))) return rc;
    k_guess<<<(unsigned)c->num_sms * 8, 256, 0, c->stream>>>(c->nL, pj->L, pj->P, pj->AP, pj->coef, b, xbar, b_reduced);
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

extern "C" int sem_proj_update(sem_proj* pj, const double* dx, int* accepted) {
    if (!pj) return SEM_EINVAL;
    sem_ctx* c = pj->c;
    c->err.clear();
    if (!dx || ((uintptr_t)dx % 16)) return sem_fail(c, SEM_EINVAL, "sem_proj_update: NULL or misaligned vector");
    int rc;
    if ((rc = sem_launch_ax_gs(c, dx, pj->w, SEM_F64, c->lambda, nullptr, nullptr))) return rc;
    if (pj->L >= pj->Lmax) pj->L = 0;                      // restart (S27)
    if ((rc = multidot(pj, pj->P, pj->L, pj->w, dx))) return rc;       // beta_i = p_i^T A dx, gamma = dx^T A dx
    k_append<<<(unsigned)c->num_sms * 8, 256, 0, c->stream>>>(c->nL, pj->L, pj->P, pj->AP, pj->coef, dx, pj->w,
                                                              pj->P + (int64_t)pj->L * c->nL,
                                                              pj->AP + (int64_t)pj->L * c->nL, pj->flag);
    int h = 0;
    SEM_CUDA_OK(c, cudaMemcpyAsync(&h, pj->flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    SEM_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    SEM_CUDA_OK(c, cudaGetLastError());
    if (h) ++pj->L;
    if (accepted) *accepted = h;
    return SEM_OK;
}

extern "C" int sem_proj_size(sem_proj* pj, int* L) {
    if (!pj || !L) return SEM_EINVAL;
    *L = pj->L;
    return SEM_OK;
}

extern "C" void sem_proj_destroy(sem_proj* pj) {
    if (!pj) return;
    if (pj->c) cudaStreamSynchronize(pj->c->stream);
    cudaFree(pj->P); cudaFree(pj->AP); cudaFree(pj->w); cudaFree(pj->coef); cudaFree(pj->flag);
    cudaGetLastError();
    delete pj;
}
