// sem_api.cu — the C ABI of include/sem.h: argument checks, context life cycle, accessors.  No arithmetic here.
#include <stdarg.h>
#include <stdio.h>

#include <new>

#include "sem_internal.h"

int sem_fail(sem_ctx* c, int code, const char* fmt, ...) {
    if (c) {
        char buf[512];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof(buf), fmt, ap);
        va_end(ap);
        c->err = buf;
    }
    cudaGetLastError();   // do not let a sticky-free error leak into the next call
    return code;
}

static int require_geom(sem_ctx* c, const char* who) {
    if (!c->geom_done) return sem_fail(c, SEM_ESTATE, "%s before sem_geom", who);
    return SEM_OK;
}

// gather-scatter (with the Dirichlet mask) of nf fields in launches of 4, 3 or 2; a single one by sem_gs's kernel
int sem_launch_gs_fields(sem_ctx* c, void* w, int nf, int64_t stride, sem_prec prec, bool mask, const int* skip) {
    const size_t vs = prec == SEM_F64 ? 8 : 4;
    for (int f = 0; f < nf;) {
        const int left = nf - f, take = left >= 4 && left != 5 ? 4 : left >= 3 ? 3 : left;
        void* wf = (char*)w + (size_t)f * (size_t)stride * vs;
        const int rc = take == 1 ? sem_launch_gs(c, wf, prec, mask, skip) : sem_launch_gs_many(c, wf, take, stride, prec, mask, skip);
        if (rc) return rc;
        f += take;
    }
    return SEM_OK;
}

int sem_mesh_setup_impl(sem_ctx** out, int64_t E, int N, const double* vertex_xyz, const int64_t* gid,
                        const uint8_t* dirichlet, void* cuda_stream, bool is_inner) {
    if (!out) return SEM_EINVAL;
    *out = nullptr;
    if (E <= 0 || N < 1 || N > SEM_MAXP - 1 || !vertex_xyz || !gid) return SEM_EINVAL;
    const int64_t p = N + 1;
    const int64_t nL = E * p * p * p;
    if (nL >= ((int64_t)1 << 31)) return SEM_EINVAL;
    sem_ctx* c = new (std::nothrow) sem_ctx();
    if (!c) return SEM_ENOMEM;
    *out = c;
    c->is_inner = is_inner;
    c->E = E; c->N = N; c->p = (int)p; c->p3 = p * p * p; c->nL = nL;
    c->epb = sem_epb((int)p);
    c->ngroups = (E + c->epb - 1) / c->epb;
    c->stream = (cudaStream_t)cuda_stream;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return sem_fail(c, SEM_ECUDA, "no CUDA device (libsem has no CPU fallback)");
    SEM_CUDA_OK(c, cudaGetDevice(&c->device));
    SEM_CUDA_OK(c, cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device));
    sem_gll_tables(N, c->xi, c->rho, c->D);
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_vert, E * 24 * sizeof(double)));
    SEM_CUDA_OK(c, cudaMemcpyAsync(c->d_vert, vertex_xyz, E * 24 * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    int rc = sem_build_maps(c, gid, dirichlet);
    if (rc) return rc;
    return sem_build_gs_records(c);
}

extern "C" {

int sem_mesh_setup(sem_ctx** out, int64_t E, int N, const double* vertex_xyz, const int64_t* gid,
                   const uint8_t* dirichlet, void* cuda_stream) {
    return sem_mesh_setup_impl(out, E, N, vertex_xyz, gid, dirichlet, cuda_stream, false);
}

int sem_geom(sem_ctx* c, const double* node_xyz, sem_gmode mode, int with_mass) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (mode != SEM_G_STORED && mode != SEM_G_RECOMPUTE) return sem_fail(c, SEM_EINVAL, "bad sem_gmode");
    if (!c->d_l2u) return sem_fail(c, SEM_ESTATE, "sem_geom on a context whose setup failed");
    if (mode == SEM_G_RECOMPUTE && node_xyz)
        return sem_fail(c, SEM_ESTATE, "SEM_G_RECOMPUTE needs trilinear geometry (node_xyz == NULL)");
    c->geom_done = false;
    sem_schwarz_free(c);        // the Schwarz smoother's factorisations belong to the geometry (and are baked into graphs)
    sem_coarse_free(c);         // so does the assembled coarse operator
    ++c->generation;
    c->pcg_ready = false;
    c->lambda_of_diag = -1.0;   // invalidates the Jacobi diagonal (lambda >= 0 always)
    c->gmode = mode;
    c->with_mass = with_mass != 0;
    int rc = sem_build_geom(c, node_xyz);
    if (rc) return rc;
    c->geom_done = true;
    return sem_inner_build(c, node_xyz);          // large mesh in an order without locality: inner context for sem_pcg
}

static int check_vec(sem_ctx* c, const void* u, const void* w, sem_prec prec, double lambda, const char* who) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (!w || (!u && who[4] == 'a')) return sem_fail(c, SEM_EINVAL, "%s: NULL vector", who);
    if (prec != SEM_F64 && prec != SEM_F32) return sem_fail(c, SEM_EINVAL, "%s: bad sem_prec", who);
    const size_t al = prec == SEM_F64 ? 8 : 4;
    if (((uintptr_t)w % al) || (u && ((uintptr_t)u % al))) return sem_fail(c, SEM_EINVAL, "%s: misaligned vector", who);
    if (u == w) return sem_fail(c, SEM_EINVAL, "%s: u and w must not alias", who);
    if (lambda != 0.0 && !c->with_mass) return sem_fail(c, SEM_ESTATE, "%s: lambda != 0 needs with_mass", who);
    return SEM_OK;
}

int sem_ax(sem_ctx* c, const void* u, void* w, sem_prec prec, double lambda) {
    int rc = check_vec(c, u, w, prec, lambda, "sem_ax");
    if (rc) return rc;
    if ((rc = require_geom(c, "sem_ax"))) return rc;
    if (prec == SEM_F32 && (rc = sem_build_g32(c))) return rc;
    return sem_launch_ax(c, u, w, prec, lambda, nullptr, nullptr);
}

int sem_gs(sem_ctx* c, void* w, sem_prec prec, sem_op op) {
    int rc = check_vec(c, nullptr, w, prec, 0.0, "sem_gs");
    if (rc) return rc;
    if (op != SEM_OP_ADD) return sem_fail(c, SEM_EINVAL, "sem_gs: only SEM_OP_ADD is defined (P:119)");
    if (!c->d_sh_off) return sem_fail(c, SEM_ESTATE, "sem_gs on a context whose setup failed");
    return sem_launch_gs(c, w, prec, false);
}

int sem_gs_many(sem_ctx* c, void* w, int nfields, int64_t field_stride, sem_prec prec, sem_op op) {
    int rc = check_vec(c, nullptr, w, prec, 0.0, "sem_gs_many");
    if (rc) return rc;
    if (op != SEM_OP_ADD) return sem_fail(c, SEM_EINVAL, "sem_gs_many: only SEM_OP_ADD is defined (P:119)");
    const bool inter = field_stride == SEM_INTERLEAVED;
    if (inter ? (nfields < 2 || nfields > 4) : (nfields < 1 || field_stride < c->nL))
        return sem_fail(c, SEM_EINVAL, "sem_gs_many: nfields < 1 or field_stride < nL (interleaved: 2 <= nfields <= 4)");
    if (!c->d_sh_off) return sem_fail(c, SEM_ESTATE, "sem_gs_many on a context whose setup failed");
    if (inter) return sem_launch_gs_many(c, w, nfields, 1, prec, false);
    const size_t vs = prec == SEM_F64 ? 8 : 4;
    for (int f = 0; f < nfields;) {                          // launches of 4, 3 or 2 fields; a single one by sem_gs's kernel
        const int left = nfields - f, take = left >= 4 && left != 5 ? 4 : left >= 3 ? 3 : left;
        void* wf = (char*)w + (size_t)f * (size_t)field_stride * vs;
        rc = take == 1 ? sem_launch_gs(c, wf, prec, false) : sem_launch_gs_many(c, wf, take, field_stride, prec, false);
        if (rc) return rc;
        f += take;
    }
    return SEM_OK;
}

int sem_ax_gs_many(sem_ctx* c, const void* u, void* w, int nfields, int64_t field_stride, sem_prec prec, double lambda) {
    int rc = check_vec(c, u, w, prec, lambda, "sem_ax_gs_many");
    if (rc) return rc;
    if ((rc = require_geom(c, "sem_ax_gs_many"))) return rc;
    if (nfields < 1 || field_stride < c->nL)
        return sem_fail(c, SEM_EINVAL, "sem_ax_gs_many: nfields < 1 or field_stride < nL");
    if (prec == SEM_F32 && (rc = sem_build_g32(c))) return rc;
    if ((rc = sem_launch_ax_many(c, u, w, nfields, field_stride, prec, lambda, nullptr, 0, nullptr))) return rc;
    return sem_launch_gs_fields(c, w, nfields, field_stride, prec, true, nullptr);
}

int sem_ax_gs(sem_ctx* c, const void* u, void* w, sem_prec prec, double lambda) {
    int rc = check_vec(c, u, w, prec, lambda, "sem_ax_gs");
    if (rc) return rc;
    if ((rc = require_geom(c, "sem_ax_gs"))) return rc;
    if (prec == SEM_F32 && (rc = sem_build_g32(c))) return rc;
    // Repeated applications with the same arguments (a time loop, a benchmark) replay a two-node CUDA graph: the
    // operator kernel and the gather-scatter kernel then start back to back instead of paying a stream launch each
    // (an empty 2000-CTA kernel costs 4 us per launch on this machine).  The first call with a new argument set runs
    // eagerly, the second is captured; the legacy default stream cannot be captured and stays eager.
    const bool same = c->ag_exec_or_seen && c->ag_u == u && c->ag_w == w && c->ag_prec == (int)prec &&
                      c->ag_lambda == lambda && c->ag_gen == c->generation && c->ag_variant == c->ax_variant;
    if (same && c->ag_exec) {
        SEM_CUDA_OK(c, cudaGraphLaunch(c->ag_exec, c->stream));
        return SEM_OK;
    }
    if (!same) {
        if (c->ag_exec) { cudaGraphExecDestroy(c->ag_exec); c->ag_exec = nullptr; }
        c->ag_u = u; c->ag_w = w; c->ag_prec = (int)prec; c->ag_lambda = lambda; c->ag_gen = c->generation;
        c->ag_variant = c->ax_variant;
        c->ag_exec_or_seen = true;
        c->ag_capturable = c->stream != nullptr && c->stream != cudaStreamLegacy;
        return sem_launch_ax_gs(c, u, w, prec, lambda, nullptr, nullptr);
    }
    if (!c->ag_capturable || cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();
        c->ag_capturable = false;
        return sem_launch_ax_gs(c, u, w, prec, lambda, nullptr, nullptr);
    }
    rc = sem_launch_ax_gs(c, u, w, prec, lambda, nullptr, nullptr);
    cudaGraph_t graph = nullptr;
    const cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    if (rc == SEM_OK && e == cudaSuccess && graph && cudaGraphInstantiate(&c->ag_exec, graph, 0) == cudaSuccess) {
        cudaGraphDestroy(graph);
        SEM_CUDA_OK(c, cudaGraphLaunch(c->ag_exec, c->stream));
        return SEM_OK;
    }
    if (graph) cudaGraphDestroy(graph);
    cudaGetLastError();
    c->ag_exec = nullptr;
    c->ag_capturable = false;
    return rc != SEM_OK ? rc : sem_launch_ax_gs(c, u, w, prec, lambda, nullptr, nullptr);
}

int sem_set_lambda(sem_ctx* c, double lambda) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (!(lambda >= 0.0)) return sem_fail(c, SEM_EINVAL, "lambda must be >= 0 (S18)");
    if (lambda != 0.0 && c->geom_done && !c->with_mass) return sem_fail(c, SEM_ESTATE, "lambda != 0 needs with_mass");
    if (c->lambda != lambda) ++c->generation;
    c->lambda = lambda;
    return SEM_OK;
}

int sem_set_variant(sem_ctx* c, int ax_variant) {
    if (!c) return SEM_EINVAL;
    if (ax_variant >= 100) c->fdm_variant = ax_variant - 100;      // 100 + v: the local-solve kernel (sem_fdm.cu)
    else c->ax_variant = ax_variant;
    return SEM_OK;
}

int sem_get_pcg_history(sem_ctx* c, double* hist, int n) {
    if (!c || !hist || n < 0) return SEM_EINVAL;
    for (int i = 0; i < n && i < c->hist_n; ++i) hist[i] = c->h_hist[i];
    return SEM_OK;
}

int sem_get_counts(sem_ctx* c, int64_t* nL, int64_t* U, int64_t* S, int64_t* Us) {
    if (!c) return SEM_EINVAL;
    if (nL) *nL = c->nL;
    if (U) *U = c->U;
    if (S) *S = c->S;
    if (Us) *Us = c->Us;
    return SEM_OK;
}

int sem_get_maps(sem_ctx* c, int32_t* l2u, int32_t* mult, int64_t* seg_off, int32_t* seg_idx, int64_t* uniq_gid) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (!c->d_l2u || !c->d_sh_off) return sem_fail(c, SEM_ESTATE, "maps not built");
    cudaStream_t st = c->stream;
    if (l2u) SEM_CUDA_OK(c, cudaMemcpyAsync(l2u, c->d_l2u, c->nL * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    if (mult) SEM_CUDA_OK(c, cudaMemcpyAsync(mult, c->d_mult, c->U * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    if (seg_off) SEM_CUDA_OK(c, cudaMemcpyAsync(seg_off, c->d_seg_off, (c->U + 1) * sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    if (seg_idx) SEM_CUDA_OK(c, cudaMemcpyAsync(seg_idx, c->d_seg_idx, c->nL * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    if (uniq_gid) SEM_CUDA_OK(c, cudaMemcpyAsync(uniq_gid, c->d_uniq_gid, c->U * sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    return SEM_OK;
}

int sem_get_gll(sem_ctx* c, double* xi, double* rho, double* D) {
    if (!c) return SEM_EINVAL;
    for (int i = 0; i < c->p; ++i) { if (xi) xi[i] = c->xi[i]; if (rho) rho[i] = c->rho[i]; }
    if (D) for (int q = 0; q < c->p * c->p; ++q) D[q] = c->D[q];
    return SEM_OK;
}

int sem_get_geom(sem_ctx* c, double* G, double* detJ) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    int rc = require_geom(c, "sem_get_geom");
    if (rc) return rc;
    return sem_geom_export(c, G, detJ);
}

int sem_get_diag(sem_ctx* c, double* diagA_local) {
    if (!c || !diagA_local) return SEM_EINVAL;
    c->err.clear();
    int rc = require_geom(c, "sem_get_diag");
    if (rc) return rc;
    if (c->lambda != 0.0 && !c->with_mass) return sem_fail(c, SEM_ESTATE, "lambda != 0 needs with_mass");
    if (!c->d_diag || c->lambda_of_diag != c->lambda) {
        if ((rc = sem_build_diag(c))) return rc;
    }
    SEM_CUDA_OK(c, cudaMemcpyAsync(diagA_local, c->d_diag, c->nL * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    SEM_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    return SEM_OK;
}

const char* sem_last_error(sem_ctx* c) {
    if (!c) return "no context (allocation failed or invalid arguments)";
    return c->err.c_str();
}

void sem_ctx_destroy(sem_ctx* c) {
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    if (c->ag_exec) cudaGraphExecDestroy(c->ag_exec);
    sem_inner_free(c);
    sem_schwarz_free(c);
    sem_coarse_free(c);
    void* ptrs[] = {c->d_vert, c->d_l2u, c->d_mult, c->d_seg_off, c->d_seg_idx, c->d_uniq_gid, c->d_sh_off, c->d_sh_idx,
                    c->d_sh_masked, c->d_mask_u, c->d_mask1_idx, c->d_G, c->d_G32, c->d_B, c->d_B32, c->d_detJ,
                    c->d_diag, c->d_Minv, c->d_wt, c->d_wt8, c->d_r, c->d_p, c->d_w, c->d_scal, 
                    c->d_own_pair, c->d_own_quad, c->d_own_big, c->d_J, c->d_cheb[0], c->d_cheb[1], c->d_cheb[2], c->d_cheb4, c->d_Minv32, c->d_Minv_g, c->d_wt_g};
    for (void* p : ptrs) cudaFree(p);
    cudaGetLastError();
    delete[] c->h_hist;
    delete c;
}

}  // extern "C"
