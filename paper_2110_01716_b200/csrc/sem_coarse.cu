// sem_coarse.cu — the coarsest p-multigrid level (N = 1) with an ASSEMBLED operator.
// P:181 (and Table 2's gs rows) say of the paper's coarse levels what ncu says of ours: at N = 1 a level of 7200 elements
// has 8379 unique nodes and every kernel on it is pure launch latency -- one Chebyshev-Jacobi step is three launches
// (operator 3 us, gather-scatter 5 us, vector update 3 us) for 0.2 MB of data, and the coarse solve of a V-cycle is 8 such
// steps.  (The paper hands this level to an algebraic multigrid solver on the CPUs; out of scope, S25.)
// Here the N = 1 operator M QQ^T (D^T G D + lambda B) M is assembled once into a sparse matrix (<= 27 entries per row
// on a hexahedral mesh) and a whole Chebyshev step -- w = A d, x += d, r -= Minv w, d' = c1 d + c2 r -- is ONE kernel
// with one thread per LOCAL node: every copy of a unique node evaluates the same row in the same order, so the field
// stays continuous bit for bit and no gather-scatter is needed; d is double-buffered because the row reads the
// neighbours' d.  Same recurrence and scalars as sem_cheby.cu (S23); only the summation order inside A d differs from
// the matrix-free operator (round-off).
#include <math.h>

#include <map>
#include <vector>

#include "sem_internal.h"

struct sem_coarse_data {
    int32_t* d_row_off = nullptr;     // [U+1]
    int32_t* d_col = nullptr;         // [nnz] local index of the FIRST copy of the column's unique node
    double* d_val64 = nullptr;
    float* d_val32 = nullptr;
    void* d_d2 = nullptr;             // second d buffer (nL doubles)
    double lambda_of = -1.0;
    int64_t nnz = 0;
};

void sem_coarse_free(sem_ctx* c) {
    sem_coarse_data* s = c->coarse;
    if (!s) return;
    cudaFree(s->d_row_off); cudaFree(s->d_col); cudaFree(s->d_val64); cudaFree(s->d_val32); cudaFree(s->d_d2);
    cudaGetLastError();
    delete s;
    c->coarse = nullptr;
}

bool sem_coarse_is_current(const sem_ctx* c) { return c->coarse && c->coarse->lambda_of == c->lambda; }

namespace {

__global__ void k_basis(int64_t n, int p3, int i, double* __restrict__ u) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x)
        u[l] = (l % p3) == i ? 1.0 : 0.0;
}

template <typename T>
__device__ __forceinline__ T row_dot(const int32_t* __restrict__ row_off, const int32_t* __restrict__ col,
                                     const T* __restrict__ val, int32_t g, const T* __restrict__ x) {
    T s = T(0);
    for (int32_t q = row_off[g]; q < row_off[g + 1]; ++q) s += val[q] * x[col[q]];
    return s;
}

// w = A x (the residual of a non-zero initial guess)
template <typename T>
__global__ void __launch_bounds__(256) k_csr_apply(int64_t n, const int32_t* __restrict__ l2u,
                                                   const int32_t* __restrict__ row_off, const int32_t* __restrict__ col,
                                                   const T* __restrict__ val, const T* __restrict__ x, T* __restrict__ w) {
    const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (l < n) w[l] = row_dot<T>(row_off, col, val, l2u[l], x);
}

// one Chebyshev step (sem_cheby.cu's k_cheb_step with the operator inside): din -> dout
template <typename T, bool XZERO, bool LAST>
__global__ void __launch_bounds__(256) k_csr_step(int64_t n, const int32_t* __restrict__ l2u,
                                                  const int32_t* __restrict__ row_off, const int32_t* __restrict__ col,
                                                  const T* __restrict__ val, const T* __restrict__ Minv, T c1, T c2,
                                                  T* __restrict__ x, T* __restrict__ r, const T* __restrict__ din,
                                                  T* __restrict__ dout) {
    const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (l >= n) return;
    const T w = row_dot<T>(row_off, col, val, l2u[l], din);
    const T dl = din[l];
    const T rl = r[l] - Minv[l] * w;
    const T dn = c1 * dl + c2 * rl;
    const T x0 = XZERO ? T(0) : x[l];
    if constexpr (LAST) {
        x[l] = x0 + dl + dn;
    } else {
        x[l] = x0 + dl;
        r[l] = rl;
        dout[l] = dn;
    }
}

// r = Minv (b - q); d = r / theta; ONLY (order 1): x <- x0 + d
template <typename T, bool ONLY>
__global__ void __launch_bounds__(256) k_csr_first(int64_t n, const T* __restrict__ b, const T* __restrict__ q,
                                                   const T* __restrict__ Minv, T inv_theta, T* __restrict__ x,
                                                   T* __restrict__ r, T* __restrict__ d) {
    const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (l >= n) return;
    const T m = Minv[l];
    const T rl = m * (q ? b[l] - q[l] : b[l]);
    const T dl = rl * inv_theta;
    if constexpr (ONLY) x[l] = (q && m != T(0)) ? x[l] + dl : dl;
    else { r[l] = rl; d[l] = dl; }
}

template <typename T>
__global__ void __launch_bounds__(256) k_csr_mask(int64_t n, const T* __restrict__ Minv, T* __restrict__ x) {
    const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (l < n && Minv[l] == T(0)) x[l] = T(0);
}

}  // namespace

// Assemble M QQ^T (D^T G D + lambda B) M for an N = 1 context: 8 operator applications on the element-local unit vectors
// give every element matrix; rows are summed over the copies of a unique node on the host.
int sem_coarse_build(sem_ctx* c) {
    if (c->coarse && c->coarse->lambda_of == c->lambda) return SEM_OK;
    sem_coarse_free(c);
    if (c->p != 2) return sem_fail(c, SEM_EINVAL, "assembled coarse operator: N = 1 only");
    cudaStream_t st = c->stream;
    const int64_t n = c->nL, E = c->E, U = c->U;
    double *d_u = nullptr, *d_w = nullptr;
    SEM_CUDA_OK(c, cudaMalloc((void**)&d_u, n * sizeof(double)));
    SEM_CUDA_OK(c, cudaMalloc((void**)&d_w, n * sizeof(double)));
    std::vector<double> Ae((size_t)E * 64), col(n);
    int rc = SEM_OK;
    for (int i = 0; i < 8 && rc == SEM_OK; ++i) {
        k_basis<<<(unsigned)c->num_sms * 4, 256, 0, st>>>(n, 8, i, d_u);
        rc = sem_launch_ax(c, d_u, d_w, SEM_F64, c->lambda, nullptr, nullptr);
        if (rc) break;
        if (cudaMemcpyAsync(col.data(), d_w, n * sizeof(double), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
            cudaStreamSynchronize(st) != cudaSuccess)
            rc = sem_fail(c, SEM_ECUDA, "assembled coarse operator: copy failed");
        for (int64_t e = 0; e < E && rc == SEM_OK; ++e)
            for (int r = 0; r < 8; ++r) Ae[(e * 8 + r) * 8 + i] = col[e * 8 + r];       // A_e[r][i]
    }
    cudaFree(d_u);
    cudaFree(d_w);
    if (rc) return rc;
    std::vector<int32_t> l2u(n), seg_idx(n);
    std::vector<int64_t> seg_off(U + 1);
    std::vector<uint8_t> mask_u(c->has_mask ? U : 0);
    SEM_CUDA_OK(c, cudaMemcpyAsync(l2u.data(), c->d_l2u, n * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaMemcpyAsync(seg_idx.data(), c->d_seg_idx, n * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaMemcpyAsync(seg_off.data(), c->d_seg_off, (U + 1) * sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    if (c->has_mask) SEM_CUDA_OK(c, cudaMemcpyAsync(mask_u.data(), c->d_mask_u, U, cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    std::vector<int32_t> row_off(U + 1, 0), cols;
    std::vector<double> vals;
    std::map<int32_t, double> row;
    for (int64_t g = 0; g < U; ++g) {
        row.clear();
        if (!(c->has_mask && mask_u[g])) {
            for (int64_t q = seg_off[g]; q < seg_off[g + 1]; ++q) {                  // copies in ascending local index
                const int64_t l = seg_idx[q], e = l / 8;
                const int r = (int)(l - e * 8);
                for (int j = 0; j < 8; ++j) {
                    const int32_t gc = l2u[e * 8 + j];
                    if (c->has_mask && mask_u[gc]) continue;
                    row[gc] += Ae[(e * 8 + r) * 8 + j];
                }
            }
        }
        for (const auto& kv : row) { cols.push_back(seg_idx[seg_off[kv.first]]); vals.push_back(kv.second); }
        row_off[g + 1] = (int32_t)cols.size();
    }
    sem_coarse_data* s = new sem_coarse_data();
    c->coarse = s;
    s->nnz = (int64_t)cols.size();
    std::vector<float> v32(vals.begin(), vals.end());
    const size_t nz = cols.size() ? cols.size() : 1;
    SEM_CUDA_OK(c, cudaMalloc((void**)&s->d_row_off, (U + 1) * sizeof(int32_t)));
    SEM_CUDA_OK(c, cudaMalloc((void**)&s->d_col, nz * sizeof(int32_t)));
    SEM_CUDA_OK(c, cudaMalloc((void**)&s->d_val64, nz * sizeof(double)));
    SEM_CUDA_OK(c, cudaMalloc((void**)&s->d_val32, nz * sizeof(float)));
    SEM_CUDA_OK(c, cudaMalloc(&s->d_d2, n * sizeof(double)));
    SEM_CUDA_OK(c, cudaMemcpyAsync(s->d_row_off, row_off.data(), (U + 1) * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    SEM_CUDA_OK(c, cudaMemcpyAsync(s->d_col, cols.data(), cols.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    SEM_CUDA_OK(c, cudaMemcpyAsync(s->d_val64, vals.data(), vals.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    SEM_CUDA_OK(c, cudaMemcpyAsync(s->d_val32, v32.data(), v32.size() * sizeof(float), cudaMemcpyHostToDevice, st));
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    s->lambda_of = c->lambda;
    return SEM_OK;
}

// sem_cheby's recurrence on the assembled operator (called by sem_cheby for N = 1 contexts once it is built)
template <typename T>
static int coarse_run(sem_ctx* c, const T* b, T* x, int order, double lmin, double lmax, bool zero_guess) {
    sem_coarse_data* s = c->coarse;
    cudaStream_t st = c->stream;
    const int64_t n = c->nL;
    T* r = (T*)c->d_cheb[0];
    T* d0 = (T*)c->d_cheb[1];
    T* w = (T*)c->d_cheb[2];
    T* d1 = (T*)s->d_d2;
    const T* Minv = sizeof(T) == 8 ? (const T*)c->d_Minv : (const T*)c->d_Minv32;
    const T* val = sizeof(T) == 8 ? (const T*)s->d_val64 : (const T*)s->d_val32;
    const unsigned grid = (unsigned)((n + 255) / 256);
    const double theta = 0.5 * (lmax + lmin), delta = 0.5 * (lmax - lmin), sigma = theta / delta;
    double rho = 1.0 / sigma;
    const T* q = nullptr;
    if (!zero_guess) {
        k_csr_mask<T><<<grid, 256, 0, st>>>(n, Minv, x);
        k_csr_apply<T><<<grid, 256, 0, st>>>(n, c->d_l2u, s->d_row_off, s->d_col, val, x, w);
        q = w;
    }
    if (order == 1) k_csr_first<T, true><<<grid, 256, 0, st>>>(n, b, q, Minv, (T)(1.0 / theta), x, r, d0);
    else k_csr_first<T, false><<<grid, 256, 0, st>>>(n, b, q, Minv, (T)(1.0 / theta), x, r, d0);
    T *din = d0, *dout = d1;
    for (int k = 1; k < order; ++k) {
        const double rho1 = 1.0 / (2.0 * sigma - rho);
        const T c1 = (T)(rho1 * rho), c2 = (T)(2.0 * rho1 / delta);
        const bool xzero = zero_guess && k == 1, last = k == order - 1;
#define SEM_CSR_STEP(XZ, LA) \
    k_csr_step<T, XZ, LA><<<grid, 256, 0, st>>>(n, c->d_l2u, s->d_row_off, s->d_col, val, Minv, c1, c2, x, r, din, dout)
        if (xzero && last) SEM_CSR_STEP(true, true);
        else if (xzero) SEM_CSR_STEP(true, false);
        else if (last) SEM_CSR_STEP(false, true);
        else SEM_CSR_STEP(false, false);
#undef SEM_CSR_STEP
        T* t = din; din = dout; dout = t;
        rho = rho1;
    }
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

int sem_coarse_cheby(sem_ctx* c, const void* b, void* x, int order, double lmin, double lmax, bool zero_guess,
                     sem_prec prec) {
    if (prec == SEM_F64) return coarse_run<double>(c, (const double*)b, (double*)x, order, lmin, lmax, zero_guess);
    return coarse_run<float>(c, (const float*)b, (float*)x, order, lmin, lmax, zero_guess);
}
