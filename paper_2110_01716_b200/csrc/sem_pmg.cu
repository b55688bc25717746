// sem_pmg.cu — NEXT-1c: one p-multigrid V-cycle as a preconditioner application z = M^-1 r.
// P:103 "p-multigrid (pMG) preconditioning ... Coarse-to-fine interpolations are cast as efficient tensor contractions
// ... Smoothers for pMG include Chebyshev-accelerated point-Jacobi"; "all steps of pMG in 32-bit arithmetic";
// P:146 level schedules.  The paper lists the ingredients, not the cycle; the reading (S25) is
//   coarsest level:  z = Chebyshev-Jacobi(A, r, coarse_order steps, zero guess)     (stands in for the paper's AMG solve)
//   otherwise:       z   = smooth(A, r, zero guess)
//                    res = r - A z
//                    r_c = M_c Q_c Q_c^T J^T (W res)      W = 1/multiplicity on the local copies (un-assembly)
//                    z  += J e_c,  e_c = vcycle(r_c)
//                    z   = smooth(A, r, guess z)
// Every level is its own context (its own discretisation of order N_l on the same elements, S17).  Host code only
// sequences kernels that exist (sem_cheby, sem_ax_gs, sem_transfer with the weighted residual / the correction update
// fused into its load / store, sem_gs); no synchronisation anywhere in the cycle.
#include <math.h>

#include <new>
#include <vector>

#include "sem_internal.h"

struct sem_pmg {
    std::vector<sem_ctx*> lv;
    std::vector<double> lmin, lmax;
    int smooth_order = 2, coarse_order = 8;
    sem_prec prec = SEM_F32;
    sem_smoother smoother = SEM_SMOOTH_CHEBY_JACOBI;
    std::vector<double> slmin, slmax;   // bounds of S A per level for the Schwarz smoothers
    std::vector<void*> r, z, w;         // per level work vectors (r, z below the finest; w above the coarsest)
    // flexible PCG (sem_fpcg): FP64 outer vectors on the finest level, FP32 copies for an FP32 cycle, 4 device scalars
    double* f[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};      // r, p, q, z, zold
    float* f32[2] = {nullptr, nullptr};                                // r, z in the cycle's precision
    double* fs = nullptr;
    std::vector<double> hist;
    // CUDA graph of one cycle for the (r, z) pair it was captured with; calls = eager cycles run with that pair so far
    const void* g_r = nullptr;
    void* g_z = nullptr;
    int g_calls = 0;
    uint64_t g_gen = 0;                 // sum of the levels' generations when the graph was recorded
    cudaGraphExec_t g_exec = nullptr;
    // CUDA graph of one whole flexible-PCG iteration (cycle, direction, operator, update), for the x it was recorded with
    bool outer_capture = false;         // the cycle is being recorded as part of that graph: run it eagerly
    cudaGraphExec_t it_exec = nullptr;
    const void* it_x = nullptr;
    const void* it_b = nullptr;
    uint64_t it_gen = 0;
};

namespace {

// pre-/post-smoothing of level l: Chebyshev-Jacobi, or Chebyshev-Schwarz on the levels that can carry it (N >= 2)
template <typename T>
int smooth(sem_pmg* mg, int l, const T* r, T* z, int zero_guess) {
    sem_ctx* c = mg->lv[l];
    if (mg->smoother != SEM_SMOOTH_CHEBY_JACOBI && c->N >= 2)
        return sem_cheby_schwarz(c, r, z, mg->smooth_order, mg->slmin[l], mg->slmax[l], zero_guess, mg->prec,
                                 mg->smoother == SEM_SMOOTH_CHEBY_RAS ? SEM_SCHWARZ_RAS : SEM_SCHWARZ_ASM);
    return sem_cheby(c, r, z, mg->smooth_order, mg->lmin[l], mg->lmax[l], zero_guess, mg->prec);
}

template <typename T>
int cycle(sem_pmg* mg, int l, const T* r, T* z) {
    sem_ctx* c = mg->lv[l];
    const int last = (int)mg->lv.size() - 1;
    int rc;
    if (l == last) return sem_cheby(c, r, z, mg->coarse_order, mg->lmin[l], mg->lmax[l], 1, mg->prec);
    if ((rc = smooth<T>(mg, l, r, z, 1))) return rc;
    T* w = (T*)mg->w[l];
    if ((rc = sem_launch_ax_gs(c, z, w, mg->prec, c->lambda, nullptr, nullptr))) return rc;
    sem_ctx* cc = mg->lv[l + 1];
    T* rc_ = (T*)mg->r[l + 1];
    T* zc = (T*)mg->z[l + 1];
    // the weighted residual (r - w) W is formed while the restriction loads it, and the prolonged correction is added
    // to z (except at Dirichlet nodes) while the prolongation stores it: no extra passes over the fine level
    if ((rc = sem_launch_transfer(cc, c, r, rc_, mg->prec, SEM_RESTRICT, w, c->d_wt))) return rc;
    if ((rc = sem_launch_gs(cc, rc_, mg->prec, /*apply_mask=*/true))) return rc;
    if ((rc = cycle<T>(mg, l + 1, rc_, zc))) return rc;
    if ((rc = sem_launch_transfer(cc, c, zc, z, mg->prec, SEM_PROLONG, nullptr, c->d_wt))) return rc;
    return smooth<T>(mg, l, r, z, 0);
}

__device__ __forceinline__ void block_add(double v, double* __restrict__ out) {
    __shared__ double red[32];
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    if (warp == 0) {
        v = lane < nw ? red[lane] : 0.0;
        for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) atomicAdd(out, v);
    }
}

// x = 0; r = M b; s[0] += r.r (unique-node dot: weights wt)
__global__ void __launch_bounds__(256) k_f_init(int64_t n, const double* __restrict__ b, const double* __restrict__ wt,
                                                double* __restrict__ x, double* __restrict__ r, double* __restrict__ s) {
    double acc = 0.0;
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const double w = wt[l], rl = w != 0.0 ? b[l] : 0.0;
        x[l] = 0.0;
        r[l] = rl;
        acc += w * rl * rl;
    }
    block_add(acc, s + 0);
}

__global__ void __launch_bounds__(256) k_d2f(int64_t n, const double* __restrict__ a, float* __restrict__ o) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x)
        o[l] = (float)a[l];
}

// z = (double) z_cycle; s[1] += r.z; s[2] += r.zold
template <typename TZ>
__global__ void __launch_bounds__(256) k_f_z(int64_t n, const TZ* __restrict__ zc, const double* __restrict__ wt,
                                             const double* __restrict__ r, const double* __restrict__ zold,
                                             double* __restrict__ z, double* __restrict__ s) {
    double a1 = 0.0, a2 = 0.0;
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const double zl = (double)zc[l], w = wt[l] * r[l];
        z[l] = zl;
        a1 += w * zl;
        a2 += w * zold[l];
    }
    block_add(a1, s + 1);
    block_add(a2, s + 2);
}

// Device scalars s[]: 0 r.r | 1 r.z_new | 2 r.z_old | 3 p.q | 4 r_old.z_old (kept across iterations) | 5 breakdown flag
// p = z + beta p with beta = (s1 - s2) / s4 (Polak-Ribiere; 0 on the first call: s4 == 0);  zold = z
__global__ void __launch_bounds__(256) k_f_p(int64_t n, const double* __restrict__ z, double* __restrict__ p,
                                             double* __restrict__ zold, const double* __restrict__ s) {
    const double beta = s[4] != 0.0 ? (s[1] - s[2]) / s[4] : 0.0;
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const double zl = z[l];
        p[l] = zl + beta * p[l];
        zold[l] = zl;
    }
}

// after k_f_p: r.z of this iteration becomes the "old" one, the accumulators are cleared for the next iteration
__global__ void k_f_roll(double* __restrict__ s) {
    s[4] = s[1];
    s[0] = s[1] = s[2] = s[3] = 0.0;
}

// x += alpha p; r -= alpha q with alpha = s4 / s3 (p.q <= 0: breakdown, nothing is changed, s5 = 1); s[0] += r.r
__global__ void __launch_bounds__(256) k_f_update(int64_t n, const double* __restrict__ p, const double* __restrict__ q,
                                                  const double* __restrict__ wt, double* __restrict__ x,
                                                  double* __restrict__ r, double* __restrict__ s) {
    const double pq = s[3];
    if (!(pq > 0.0)) {
        if (blockIdx.x == 0 && threadIdx.x == 0) s[5] = 1.0;
        return;
    }
    const double alpha = s[4] / pq;
    double acc = 0.0;
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        x[l] += alpha * p[l];
        const double rl = r[l] - alpha * q[l];
        r[l] = rl;
        acc += wt[l] * rl * rl;
    }
    block_add(acc, s + 0);
}

}  // namespace

// Flexible PCG on the finest level with the V-cycle as preconditioner (reading S26): the recurrence of O8 with the
// Polak-Ribiere beta = r_new.(z_new - z_old) / (r_old.z_old), FP64 outer iteration, cycle in mg's precision.
// alpha and beta are formed on the device; the host reads ||r||^2 once per iteration for the stopping test.
extern "C" int sem_fpcg(sem_pmg* mg, const double* b, double* x, double tol, int maxit, int* iters_out,
                        double* relres_out) {
    if (!mg) return SEM_EINVAL;
    sem_ctx* c = mg->lv[0];
    c->err.clear();
    if (!b || !x || b == x) return sem_fail(c, SEM_EINVAL, "sem_fpcg: NULL or aliased vectors");
    if (((uintptr_t)x % 16) || ((uintptr_t)b % 8)) return sem_fail(c, SEM_EINVAL, "sem_fpcg: x must be 16-byte aligned");
    if (!(tol > 0.0) && maxit <= 0) return sem_fail(c, SEM_EINVAL, "sem_fpcg: tol <= 0 with maxit <= 0");
    if (maxit < 0) maxit = 0;
    cudaStream_t st = c->stream;
    const int64_t n = c->nL;
    for (int q = 0; q < 5; ++q)
        if (!mg->f[q]) SEM_CUDA_OK(c, cudaMalloc((void**)&mg->f[q], n * sizeof(double)));
    if (mg->prec == SEM_F32)
        for (int q = 0; q < 2; ++q)
            if (!mg->f32[q]) SEM_CUDA_OK(c, cudaMalloc((void**)&mg->f32[q], n * sizeof(float)));
    if (!mg->fs) SEM_CUDA_OK(c, cudaMalloc((void**)&mg->fs, 8 * sizeof(double)));
    double *r = mg->f[0], *p = mg->f[1], *q = mg->f[2], *z = mg->f[3], *zold = mg->f[4], *s = mg->fs;
    const unsigned grid = (unsigned)c->num_sms * 8;
    double h[8];
    auto fetch = [&]() -> int {
        SEM_CUDA_OK(c, cudaMemcpyAsync(h, s, sizeof(h), cudaMemcpyDeviceToHost, st));
        SEM_CUDA_OK(c, cudaStreamSynchronize(st));
        return SEM_OK;
    };
    auto precondition = [&]() -> int {                 // z = M^-1 r, s[1] = r.z, s[2] = r.zold
        int rc;
        if (mg->prec == SEM_F32) {
            k_d2f<<<grid, 256, 0, st>>>(n, r, mg->f32[0]);
            if ((rc = sem_pmg_vcycle(mg, mg->f32[0], mg->f32[1]))) return rc;
            k_f_z<float><<<grid, 256, 0, st>>>(n, mg->f32[1], c->d_wt, r, zold, z, s);
        } else {
            if ((rc = sem_pmg_vcycle(mg, r, q))) return rc;           // q is free here
            k_f_z<double><<<grid, 256, 0, st>>>(n, q, c->d_wt, r, zold, z, s);
        }
        return SEM_OK;
    };
    mg->hist.clear();
    int rc;
    SEM_CUDA_OK(c, cudaMemsetAsync(s, 0, 8 * sizeof(double), st));
    SEM_CUDA_OK(c, cudaMemsetAsync(zold, 0, n * sizeof(double), st));
    SEM_CUDA_OK(c, cudaMemsetAsync(p, 0, n * sizeof(double), st));
    k_f_init<<<grid, 256, 0, st>>>(n, b, c->d_wt, x, r, s);
    if ((rc = fetch())) return rc;
    const double rr0 = h[0];
    int it = 0;
    mg->hist.push_back(rr0 > 0.0 ? 1.0 : 0.0);
    if (rr0 > 0.0 && maxit > 0) {
        // alpha and beta are formed on the device from the scalar slots; the host only reads ||r||^2 (and the
        // breakdown flag) once per iteration for the stopping test
        // Every launch of an iteration has the same arguments (the scalars live on the device), so from the second
        // iteration on the whole iteration is one CUDA graph (recorded once per x; non-default streams only).
        auto body = [&]() -> int {
            int rb;
            if ((rb = precondition())) return rb;                    // z, s1 = r.z, s2 = r.zold
            k_f_p<<<grid, 256, 0, st>>>(n, z, p, zold, s);
            k_f_roll<<<1, 1, 0, st>>>(s);
            if ((rb = sem_launch_ax_gs(c, p, q, SEM_F64, c->lambda, s + 3, nullptr))) return rb;
            k_f_update<<<grid, 256, 0, st>>>(n, p, q, c->d_wt, x, r, s);
            return SEM_OK;
        };
        uint64_t gen = 0;
        for (sem_ctx* lv : mg->lv) gen += lv->generation;
        if (mg->it_exec && (mg->it_x != x || mg->it_b != b || mg->it_gen != gen)) {
            cudaGraphExecDestroy(mg->it_exec);
            mg->it_exec = nullptr;
        }
        bool capturable = st != nullptr && st != cudaStreamLegacy;
        while (it < maxit) {
            if (mg->it_exec) {
                SEM_CUDA_OK(c, cudaGraphLaunch(mg->it_exec, st));
            } else if (it >= 1 && capturable && cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
                mg->outer_capture = true;
                rc = body();
                mg->outer_capture = false;
                cudaGraph_t graph = nullptr;
                const cudaError_t e = cudaStreamEndCapture(st, &graph);
                if (rc == SEM_OK && e == cudaSuccess && graph && cudaGraphInstantiate(&mg->it_exec, graph, 0) == cudaSuccess) {
                    cudaGraphDestroy(graph);
                    mg->it_x = x; mg->it_b = b; mg->it_gen = gen;
                    SEM_CUDA_OK(c, cudaGraphLaunch(mg->it_exec, st));
                } else {
                    if (graph) cudaGraphDestroy(graph);
                    cudaGetLastError();
                    mg->it_exec = nullptr;
                    capturable = false;
                    if (rc != SEM_OK) return rc;
                    if ((rc = body())) return rc;
                }
            } else {
                if (it >= 1) { cudaGetLastError(); capturable = false; }
                if ((rc = body())) return rc;
            }
            if ((rc = fetch())) return rc;
            if (h[5] != 0.0) break;                                  // breakdown (S13): x unchanged by this iteration
            ++it;
            mg->hist.push_back(sqrt(h[0] / rr0));
            if (h[0] <= tol * tol * rr0) break;
        }
    }
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    SEM_CUDA_OK(c, cudaGetLastError());
    if (iters_out) *iters_out = it;
    if (relres_out) *relres_out = mg->hist.back();
    return SEM_OK;
}

extern "C" int sem_pmg_get_history(sem_pmg* mg, double* hist, int n) {
    if (!mg || !hist || n < 0) return SEM_EINVAL;
    for (int i = 0; i < n && i < (int)mg->hist.size(); ++i) hist[i] = mg->hist[i];
    return SEM_OK;
}

extern "C" int sem_pmg_create(sem_pmg** out, int nlevels, sem_ctx* const* levels, const double* lmin,
                              const double* lmax, int smooth_order, int coarse_order, sem_prec prec) {
    if (!out) return SEM_EINVAL;
    *out = nullptr;
    if (nlevels < 1 || !levels || !lmin || !lmax || smooth_order < 1 || coarse_order < 1) return SEM_EINVAL;
    if (prec != SEM_F64 && prec != SEM_F32) return SEM_EINVAL;
    for (int l = 0; l < nlevels; ++l) {
        sem_ctx* c = levels[l];
        if (!c || !c->geom_done) return SEM_ESTATE;
        if (!(lmin[l] > 0.0) || !(lmax[l] > lmin[l])) return sem_fail(c, SEM_EINVAL, "sem_pmg_create: bad eigenvalue bounds");
        if (l > 0 && (c->E != levels[0]->E || c->N >= levels[l - 1]->N || c->stream != levels[0]->stream ||
                      c->has_mask != levels[0]->has_mask))
            return sem_fail(c, SEM_EINVAL, "sem_pmg_create: levels need equal E, stream and mask use, decreasing order");
    }
    sem_pmg* mg = new (std::nothrow) sem_pmg();
    if (!mg) return SEM_ENOMEM;
    mg->smooth_order = smooth_order;
    mg->coarse_order = coarse_order;
    mg->prec = prec;
    const size_t es = prec == SEM_F64 ? 8 : 4;
    for (int l = 0; l < nlevels; ++l) {
        sem_ctx* c = levels[l];
        mg->lv.push_back(c);
        mg->lmin.push_back(lmin[l]);
        mg->lmax.push_back(lmax[l]);
        void *r = nullptr, *z = nullptr, *w = nullptr;
        cudaError_t e = cudaSuccess;
        if (l > 0) { e = cudaMalloc(&r, c->nL * es); if (e == cudaSuccess) e = cudaMalloc(&z, c->nL * es); }
        if (e == cudaSuccess && l < nlevels - 1) e = cudaMalloc(&w, c->nL * es);
        mg->r.push_back(r); mg->z.push_back(z); mg->w.push_back(w);
        if (e != cudaSuccess) {
            sem_fail(c, SEM_ENOMEM, "sem_pmg_create: %s", cudaGetErrorString(e));
            sem_pmg_destroy(mg);
            return SEM_ENOMEM;
        }
        int rc = sem_build_diag(c);                       // wt (and Minv) are needed by the cycle's vector kernels
        if (rc) { sem_pmg_destroy(mg); return rc; }
    }
    *out = mg;
    return SEM_OK;
}

extern "C" int sem_pmg_set_smoother(sem_pmg* mg, sem_smoother smoother, const double* lmin, const double* lmax) {
    if (!mg) return SEM_EINVAL;
    sem_ctx* c0 = mg->lv[0];
    c0->err.clear();
    if (smoother != SEM_SMOOTH_CHEBY_JACOBI && smoother != SEM_SMOOTH_CHEBY_SCHWARZ && smoother != SEM_SMOOTH_CHEBY_RAS)
        return sem_fail(c0, SEM_EINVAL, "sem_pmg_set_smoother: bad sem_smoother");
    const int nl = (int)mg->lv.size();
    if (smoother != SEM_SMOOTH_CHEBY_JACOBI) {
        if (!lmin || !lmax) return sem_fail(c0, SEM_EINVAL, "sem_pmg_set_smoother: NULL bounds");
        mg->slmin.assign(lmin, lmin + nl);
        mg->slmax.assign(lmax, lmax + nl);
        for (int l = 0; l < nl - 1; ++l) {
            sem_ctx* c = mg->lv[l];
            if (c->N < 2) continue;
            if (!(lmin[l] > 0.0) || !(lmax[l] > lmin[l])) return sem_fail(c0, SEM_EINVAL, "sem_pmg_set_smoother: bad bounds");
            int rc = sem_schwarz_setup(c);
            if (rc) return rc;
        }
    }
    mg->smoother = smoother;
    if (mg->g_exec) { cudaGraphExecDestroy(mg->g_exec); mg->g_exec = nullptr; }
    if (mg->it_exec) { cudaGraphExecDestroy(mg->it_exec); mg->it_exec = nullptr; }
    mg->g_r = nullptr; mg->g_z = nullptr; mg->g_calls = 0;
    return SEM_OK;
}

extern "C" int sem_pmg_vcycle(sem_pmg* mg, const void* r, void* z) {
    if (!mg) return SEM_EINVAL;
    sem_ctx* c = mg->lv[0];
    c->err.clear();
    if (!r || !z || r == z) return sem_fail(c, SEM_EINVAL, "sem_pmg_vcycle: NULL or aliased vectors");
    auto eager = [&]() {
        return mg->prec == SEM_F64 ? cycle<double>(mg, 0, (const double*)r, (double*)z)
                                   : cycle<float>(mg, 0, (const float*)r, (float*)z);
    };
    // A cycle is ~70 small launches and the coarse levels are pure launch latency: when the same (r, z) pair
    // comes back (a Krylov loop), the second call is captured into a CUDA graph and later calls replay it.  The first
    // call runs eagerly because it may allocate and upload (interpolation matrices, work vectors), which cannot be
    // captured.
    if (mg->outer_capture) return eager();                   // part of sem_fpcg's iteration graph
    uint64_t gen = 0;
    for (sem_ctx* lv : mg->lv) gen += lv->generation;
    if (mg->g_r != r || mg->g_z != z || mg->g_gen != gen) {       // another pair, or a level was re-built / re-parametrised
        mg->g_gen = gen;
        if (mg->g_exec) { cudaGraphExecDestroy(mg->g_exec); mg->g_exec = nullptr; }
        mg->g_r = r; mg->g_z = z; mg->g_calls = 0;
    }
    if (mg->g_exec) {
        SEM_CUDA_OK(c, cudaGraphLaunch(mg->g_exec, c->stream));
        return SEM_OK;
    }
    // (the legacy default stream cannot be captured: contexts created on it stay eager)
    if (mg->g_calls++ == 0 || mg->g_calls < 0 || c->stream == nullptr || c->stream == cudaStreamLegacy) return eager();
    cudaGraph_t graph = nullptr;
    if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();
        mg->g_calls = -1000000;
        return eager();
    }
    const int rc = eager();
    const cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    if (rc != SEM_OK || e != cudaSuccess || !graph) {      // not capturable after all: stay eager for this pair
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        mg->g_calls = -1000000;
        return rc != SEM_OK ? rc : eager();
    }
    const cudaError_t ei = cudaGraphInstantiate(&mg->g_exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ei != cudaSuccess) { mg->g_exec = nullptr; cudaGetLastError(); mg->g_calls = -1000000; return eager(); }
    SEM_CUDA_OK(c, cudaGraphLaunch(mg->g_exec, c->stream));
    return SEM_OK;
}

extern "C" void sem_pmg_destroy(sem_pmg* mg) {
    if (!mg) return;
    if (!mg->lv.empty()) cudaStreamSynchronize(mg->lv[0]->stream);
    for (auto* v : {&mg->r, &mg->z, &mg->w})
        for (void* p : *v) cudaFree(p);
    if (mg->g_exec) cudaGraphExecDestroy(mg->g_exec);
    if (mg->it_exec) cudaGraphExecDestroy(mg->it_exec);
    for (double* p : mg->f) cudaFree(p);
    for (float* p : mg->f32) cudaFree(p);
    cudaFree(mg->fs);
    cudaGetLastError();
    delete mg;
}
