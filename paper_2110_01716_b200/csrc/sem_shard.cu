// sem_shard.cu — NEXT-4 (A17, A18): the operator and the Jacobi-PCG set-up when the ELEMENTS are
// partitioned over several ranks, one context per rank.  P:89 "overlap of the non-local gather-scatter with the interior
// element work"; P:101 (the solver); P:119-121 (exchange-and-sum of shared interface values).
//
// The library runs every kernel; what it cannot do itself is talk to the other ranks.  The caller hands it three hooks
// (sem_shard_hooks, include/sem.h): gs_begin / gs_end bracket the exchange of the interface values of one field (pack
// and send; receive and add -- sem_iface_pack / sem_iface_add plus the transport, NCCL in paper_2110_01716_b200/
// sharded.py), allreduce sums a few device scalars over the ranks.  All three are ordered on the context's stream.
//
// Overlap: sem_shard_set_interface(ctx, nI) declares that the first nI elements of the rank are the only ones
// touching nodes shared with other ranks.  The chunk table (sem_maps.cu) then gets a boundary after those elements'
// groups; the records of that first chunk hold every shared node (a record belongs to the chunk of the node's LAST copy,
// and every copy of a shared node lies in an interface element), so after operator + gather-scatter of chunk 0 the
// rank-local sums of the interface are final:  chunk 0 -> gs_begin -> remaining chunks -> gs_end.
#include "sem_internal.h"

namespace {

__global__ void __launch_bounds__(256) k_mult_local(int64_t n, const int32_t* __restrict__ l2u,
                                                    const int32_t* __restrict__ mult, double* __restrict__ out) {
    const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (l < n) out[l] = (double)mult[l2u[l]];
}

// Minv = mask / diag, wt = mask / mult with diag and mult summed over all ranks (S12, S14, O8)
__global__ void __launch_bounds__(256) k_minv_wt_global(int64_t n, const double* __restrict__ diag_g,
                                                        const double* __restrict__ mult_g,
                                                        const int32_t* __restrict__ l2u,
                                                        const uint8_t* __restrict__ mask_u, double* __restrict__ Minv,
                                                        double* __restrict__ wt) {
    const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (l >= n) return;
    const bool masked = mask_u && mask_u[l2u[l]];
    Minv[l] = masked ? 0.0 : 1.0 / diag_g[l];
    wt[l] = masked ? 0.0 : 1.0 / mult_g[l];
}

inline unsigned nblk(int64_t n) { return (unsigned)((n + 255) / 256); }

}  // namespace

int sem_hooks_ok(sem_ctx* c, const sem_shard_hooks* h, const char* who) {
    if (!h || !h->gs_begin || !h->gs_end || !h->allreduce) return sem_fail(c, SEM_EINVAL, "%s: incomplete sem_shard_hooks", who);
    return SEM_OK;
}

// the operator + rank-local gather-scatter with the exchange started as early as the chunk table allows
int sem_launch_ax_gs_sharded(sem_ctx* c, const void* u, void* w, sem_prec prec, double lambda, double* dot_out,
                             const int* skip_flag, const sem_shard_hooks* h) {
    int rc;
    const int nch = (int)c->chunk_e0.size() - 1;
    const int ic = c->iface_chunks;
    if (ic > 0 && ic < nch) {
        if ((rc = sem_launch_ax_gs_chunks(c, u, w, prec, lambda, dot_out, skip_flag, 0, ic))) return rc;
        if (h->gs_begin(h->user, w, (int)prec)) return sem_fail(c, SEM_ECUDA, "sharded apply: gs_begin hook failed");
        if ((rc = sem_launch_ax_gs_chunks(c, u, w, prec, lambda, dot_out, skip_flag, ic, nch))) return rc;
    } else {
        if ((rc = sem_launch_ax_gs(c, u, w, prec, lambda, dot_out, skip_flag))) return rc;
        if (h->gs_begin(h->user, w, (int)prec)) return sem_fail(c, SEM_ECUDA, "sharded apply: gs_begin hook failed");
    }
    if (h->gs_end(h->user, w, (int)prec)) return sem_fail(c, SEM_ECUDA, "sharded apply: gs_end hook failed");
    return SEM_OK;
}

// Jacobi preconditioner and dot weights of the partitioned problem: the assembled diagonal and the multiplicity summed
// over the ranks through the same exchange the fields use
int sem_shard_build_diag(sem_ctx* c, const sem_shard_hooks* h) {
    cudaStream_t st = c->stream;
    int rc = sem_build_diag(c);                         // d_diag = QQ^T diag(A_L) inside the rank (unmasked)
    if (rc) return rc;
    if (!c->d_Minv_g) {
        SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_Minv_g, c->nL * sizeof(double)));
        SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_wt_g, c->nL * sizeof(double)));
    }
    double *dg = nullptr, *mg = nullptr;
    SEM_CUDA_OK(c, cudaMalloc((void**)&dg, c->nL * sizeof(double)));
    if (cudaMalloc((void**)&mg, c->nL * sizeof(double)) != cudaSuccess) {
        cudaFree(dg);
        return sem_fail(c, SEM_ENOMEM, "sem_shard_build_diag: out of device memory");
    }
    cudaMemcpyAsync(dg, c->d_diag, c->nL * sizeof(double), cudaMemcpyDeviceToDevice, st);
    k_mult_local<<<nblk(c->nL), 256, 0, st>>>(c->nL, c->d_l2u, c->d_mult, mg);
    int bad = h->gs_begin(h->user, dg, (int)SEM_F64) || h->gs_end(h->user, dg, (int)SEM_F64);
    bad = bad || h->gs_begin(h->user, mg, (int)SEM_F64) || h->gs_end(h->user, mg, (int)SEM_F64);
    if (!bad)
        k_minv_wt_global<<<nblk(c->nL), 256, 0, st>>>(c->nL, dg, mg, c->d_l2u, c->has_mask ? c->d_mask_u : nullptr,
                                                      c->d_Minv_g, c->d_wt_g);
    const cudaError_t e = cudaStreamSynchronize(st);
    cudaFree(dg);
    cudaFree(mg);
    if (bad) return sem_fail(c, SEM_ECUDA, "sem_shard_build_diag: exchange hook failed");
    if (e != cudaSuccess) return sem_fail(c, SEM_ECUDA, "sem_shard_build_diag: %s", cudaGetErrorString(e));
    SEM_CUDA_OK(c, cudaGetLastError());
    c->lambda_of_shard = c->lambda;
    return SEM_OK;
}

extern "C" int sem_shard_set_interface(sem_ctx* c, int64_t n_iface_elems) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (n_iface_elems < 0 || n_iface_elems > c->E) return sem_fail(c, SEM_EINVAL, "sem_shard_set_interface: 0 <= n <= E");
    const int64_t groups = (n_iface_elems + c->epb - 1) / c->epb;
    const bool split = n_iface_elems > 0 && groups < c->ngroups;
    sem_default_chunks(c, split ? groups : 0);
    c->iface_chunks = split ? 1 : 0;
    ++c->generation;                                    // cached graphs were captured with the old chunk table
    return SEM_OK;
}

extern "C" int sem_get_chunks(sem_ctx* c, int64_t* elem_bounds, int cap, int* n_chunks, int* iface_chunks) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    const int nch = c->chunk_e0.size() >= 3 ? (int)c->chunk_e0.size() - 1 : 1;
    if (n_chunks) *n_chunks = nch;
    if (iface_chunks) *iface_chunks = c->iface_chunks;
    if (elem_bounds) {
        if (cap < nch + 1) return sem_fail(c, SEM_EINVAL, "sem_get_chunks: need room for %d bounds", nch + 1);
        if (nch == 1) { elem_bounds[0] = 0; elem_bounds[1] = c->E; }
        else for (int q = 0; q <= nch; ++q) elem_bounds[q] = c->chunk_e0[q];
    }
    return SEM_OK;
}

extern "C" int sem_ax_gs_sharded(sem_ctx* c, const void* u, void* w, sem_prec prec, double lambda,
                                 const sem_shard_hooks* hooks) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (!u || !w || u == w) return sem_fail(c, SEM_EINVAL, "sem_ax_gs_sharded: NULL or aliased vectors");
    if (prec != SEM_F64 && prec != SEM_F32) return sem_fail(c, SEM_EINVAL, "sem_ax_gs_sharded: bad precision");
    if (!(lambda >= 0.0)) return sem_fail(c, SEM_EINVAL, "lambda must be >= 0 (S18)");
    if (!c->geom_done) return sem_fail(c, SEM_ESTATE, "sem_ax_gs_sharded before sem_geom");
    if (lambda != 0.0 && !c->with_mass) return sem_fail(c, SEM_ESTATE, "lambda != 0 needs with_mass");
    int rc = sem_hooks_ok(c, hooks, "sem_ax_gs_sharded");
    if (rc) return rc;
    if (prec == SEM_F32 && (rc = sem_build_g32(c))) return rc;
    return sem_launch_ax_gs_sharded(c, u, w, prec, lambda, nullptr, nullptr, hooks);
}
