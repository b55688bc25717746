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
// sequences kernels that exist (sem_cheby, sem_ax_gs, sem_transfer, sem_gs) plus two element-wise vector kernels; no
// synchronisation anywhere in the cycle.
#include <new>
#include <vector>

#include "sem_internal.h"

struct sem_pmg {
    std::vector<sem_ctx*> lv;
    std::vector<double> lmin, lmax;
    int smooth_order = 2, coarse_order = 8;
    sem_prec prec = SEM_F32;
    std::vector<void*> r, z, t, w;      // per level work vectors (r, z only below the finest)
};

namespace {

// t = (r - w) * wt      wt = 1/multiplicity, 0 at Dirichlet nodes
template <typename T>
__global__ void __launch_bounds__(256) k_resw(int64_t n, const T* __restrict__ r, const T* __restrict__ w,
                                              const double* __restrict__ wt, T* __restrict__ t) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x)
        t[l] = (r[l] - w[l]) * (T)wt[l];
}

// z += t except at Dirichlet nodes
template <typename T>
__global__ void __launch_bounds__(256) k_add_unmasked(int64_t n, const T* __restrict__ t, const double* __restrict__ wt,
                                                      T* __restrict__ z) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x)
        if (wt[l] != 0.0) z[l] += t[l];
}

template <typename T>
int cycle(sem_pmg* mg, int l, const T* r, T* z) {
    sem_ctx* c = mg->lv[l];
    const int last = (int)mg->lv.size() - 1;
    int rc;
    if (l == last) return sem_cheby(c, r, z, mg->coarse_order, mg->lmin[l], mg->lmax[l], 1, mg->prec);
    if ((rc = sem_cheby(c, r, z, mg->smooth_order, mg->lmin[l], mg->lmax[l], 1, mg->prec))) return rc;
    T* w = (T*)mg->w[l];
    T* t = (T*)mg->t[l];
    if ((rc = sem_launch_ax_gs(c, z, w, mg->prec, c->lambda, nullptr, nullptr))) return rc;
    const unsigned grid = (unsigned)c->num_sms * 8;
    k_resw<T><<<grid, 256, 0, c->stream>>>(c->nL, r, w, c->d_wt, t);
    sem_ctx* cc = mg->lv[l + 1];
    T* rc_ = (T*)mg->r[l + 1];
    T* zc = (T*)mg->z[l + 1];
    if ((rc = sem_transfer(cc, c, t, rc_, mg->prec, SEM_RESTRICT))) return rc;
    if ((rc = sem_launch_gs(cc, rc_, mg->prec, /*apply_mask=*/true))) return rc;
    if ((rc = cycle<T>(mg, l + 1, rc_, zc))) return rc;
    if ((rc = sem_transfer(cc, c, zc, t, mg->prec, SEM_PROLONG))) return rc;
    k_add_unmasked<T><<<grid, 256, 0, c->stream>>>(c->nL, t, c->d_wt, z);
    SEM_CUDA_OK(c, cudaGetLastError());
    return sem_cheby(c, r, z, mg->smooth_order, mg->lmin[l], mg->lmax[l], 0, mg->prec);
}

}  // namespace

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
        void *r = nullptr, *z = nullptr, *t = nullptr, *w = nullptr;
        cudaError_t e = cudaSuccess;
        if (l > 0) { e = cudaMalloc(&r, c->nL * es); if (e == cudaSuccess) e = cudaMalloc(&z, c->nL * es); }
        if (e == cudaSuccess && l < nlevels - 1) { e = cudaMalloc(&t, c->nL * es); if (e == cudaSuccess) e = cudaMalloc(&w, c->nL * es); }
        mg->r.push_back(r); mg->z.push_back(z); mg->t.push_back(t); mg->w.push_back(w);
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

extern "C" int sem_pmg_vcycle(sem_pmg* mg, const void* r, void* z) {
    if (!mg) return SEM_EINVAL;
    sem_ctx* c = mg->lv[0];
    c->err.clear();
    if (!r || !z || r == z) return sem_fail(c, SEM_EINVAL, "sem_pmg_vcycle: NULL or aliased vectors");
    if (mg->prec == SEM_F64) return cycle<double>(mg, 0, (const double*)r, (double*)z);
    return cycle<float>(mg, 0, (const float*)r, (float*)z);
}

extern "C" void sem_pmg_destroy(sem_pmg* mg) {
    if (!mg) return;
    if (!mg->lv.empty()) cudaStreamSynchronize(mg->lv[0]->stream);
    for (auto* v : {&mg->r, &mg->z, &mg->t, &mg->w})
        for (void* p : *v) cudaFree(p);
    cudaGetLastError();
    delete mg;
}
