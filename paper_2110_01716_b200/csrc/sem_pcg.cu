// sem_pcg.cu — a8: Jacobi-preconditioned conjugate gradients on A = M QQ^T (D^T G D + lambda B) M, FP64.
// P:101 "Jacobi-preconditioned conjugate gradient iteration"; O8 / S12-S14 fix the details:
//   x = M x0; r = M b - A x; z = Minv r; p = z; rho = r.z; r0 = ||r||
//   it = 1..maxit: q = A p; alpha = rho / p.q; x += alpha p; r -= alpha q; stop if ||r|| <= tol r0;
//                  z = Minv r; rho' = r.z; beta = rho'/rho; p = z + beta p
// All vectors are in local (element) layout and continuous, so a dot over unique unmasked nodes is the local sum
// weighted by wt = mask/mult; p.q is the un-assembled local dot sum_l p_l (A_L p)_l, fused into the Ax kernel.
//
// The loop never returns to the host for a scalar: every dot lands in a per-iteration slot of a device array,
// every kernel reads what it needs from there, and a device flag turns all later launches into no-ops once the
// stopping test (or p.q <= 0) fires.  The host only polls that flag every few iterations.
#include <math.h>

#include "sem_internal.h"

namespace {

// device scalars: slot(it) = 4*it + {0: p.q, 1: r.r, 2: r.z};  it = 0 holds the initial r.r and r.z
// `it` / `ticket` / `pq`: the graph-replayed loop keeps the iteration number on the device (k_pcg_direction's last block
// advances it) and the operator adds p.q into the fixed slot `pq` (k_pcg_update moves it into the iteration's slot,
// k_pcg_direction clears it): then every launch of an iteration has the same arguments and a batch is one CUDA graph
struct PcgFlags { int done; int iters; int breakdown; int it; unsigned int ticket; int pad; double pq; };

__device__ __forceinline__ void block_sum2_atomic(double a, double b, double* __restrict__ outa,
                                                  double* __restrict__ outb) {
    __shared__ double red[2][32];
    for (int o = 16; o; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    if (lane == 0) { red[0][warp] = a; red[1][warp] = b; }
    __syncthreads();
    if (warp == 0) {
        a = lane < nw ? red[0][lane] : 0.0;
        b = lane < nw ? red[1][lane] : 0.0;
        for (int o = 16; o; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); }
        if (lane == 0) { atomicAdd(outa, a); atomicAdd(outb, b); }
    }
}

// r = M (b - q) (q = A x0, may be null), x = M x, z = Minv r, p = z; accumulate r.r and r.z into slot 0
__global__ void __launch_bounds__(256) k_pcg_init(int64_t n, const double* __restrict__ b, const double* __restrict__ q,
                                                  const double* __restrict__ Minv, const double* __restrict__ wt,
                                                  double* __restrict__ x, double* __restrict__ r,
                                                  double* __restrict__ p, double* __restrict__ scal) {
    double srr = 0.0, srz = 0.0;
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const double wl = wt[l];
        const bool live = wl != 0.0;
        const double rl = live ? (q ? b[l] - q[l] : b[l]) : 0.0;
        if (!live) x[l] = 0.0;
        const double zl = Minv[l] * rl;
        r[l] = rl;
        p[l] = zl;
        srr += wl * rl * rl;
        srz += wl * rl * zl;
    }
    block_sum2_atomic(srr, srz, scal + 1, scal + 2);
}

__global__ void __launch_bounds__(256) k_mask_vec(int64_t n, const double* __restrict__ wt, double* __restrict__ x) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x)
        if (wt[l] == 0.0) x[l] = 0.0;
}

// x += alpha p; r -= alpha w; accumulate r.r and r.z (z = Minv r) into slot it
// W8: the dot weights come from wt8 (multiplicity as a byte, 0 = Dirichlet; 1 B instead of 8 B per node), wt = 1/wt8
__device__ __forceinline__ double wt_of(uint8_t m) { return m ? 1.0 / (double)m : 0.0; }

template <bool W8>
__global__ void __launch_bounds__(256) k_pcg_update(int64_t n, int it, const double* __restrict__ p,
                                                    const double* __restrict__ w, const double* __restrict__ Minv,
                                                    const double* __restrict__ wt, const uint8_t* __restrict__ wt8,
                                                    double* __restrict__ x, double* __restrict__ r,
                                                    double* __restrict__ scal, PcgFlags* __restrict__ flags) {
    if (flags->done) return;
    const bool dev_it = it < 0;                         // graph replay: iteration number and p.q live in `flags`
    if (dev_it) it = flags->it;
    const double pq = dev_it ? flags->pq : scal[4 * it + 0];
    if (dev_it && blockIdx.x == 0 && threadIdx.x == 0) scal[4 * it + 0] = pq;
    if (!(pq > 0.0)) {                                  // breakdown (S13): stop, keep x
        if (blockIdx.x == 0 && threadIdx.x == 0) { flags->breakdown = 1; flags->iters = it; }
        // `done` is raised by k_pcg_direction so that no block of this kernel can observe it half-way
        return;
    }
    const double alpha = scal[4 * (it - 1) + 2] / pq;
    double srr = 0.0, srz = 0.0;
    const int64_t n2 = n >> 1;
    const double2* p2 = reinterpret_cast<const double2*>(p);
    const double2* w2 = reinterpret_cast<const double2*>(w);
    const double2* m2 = reinterpret_cast<const double2*>(Minv);
    const double2* t2 = reinterpret_cast<const double2*>(wt);
    double2* x2 = reinterpret_cast<double2*>(x);
    double2* r2 = reinterpret_cast<double2*>(r);
    for (int64_t v = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; v < n2; v += (int64_t)gridDim.x * blockDim.x) {
        const double2 pv = p2[v], wv = w2[v], mv = m2[v];
        double2 tv;
        if constexpr (W8) {
            const uchar2 c8 = reinterpret_cast<const uchar2*>(wt8)[v];
            tv = make_double2(wt_of(c8.x), wt_of(c8.y));
        } else {
            tv = t2[v];
        }
        double2 xv = x2[v], rv = r2[v];
        xv.x += alpha * pv.x; xv.y += alpha * pv.y;
        rv.x -= alpha * wv.x; rv.y -= alpha * wv.y;
        x2[v] = xv; r2[v] = rv;
        const double ax = tv.x * rv.x * rv.x, ay = tv.y * rv.y * rv.y;
        srr += ax + ay;
        srz += ax * mv.x + ay * mv.y;
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const int64_t l = n - 1;
        x[l] += alpha * p[l];
        const double rl = r[l] - alpha * w[l];
        r[l] = rl;
        const double wl = W8 ? wt_of(wt8[l]) : wt[l];
        srr += wl * rl * rl;
        srz += wl * rl * rl * Minv[l];
    }
    block_sum2_atomic(srr, srz, scal + 4 * it + 1, scal + 4 * it + 2);
}

// stopping test, then p = Minv r + beta p
__global__ void __launch_bounds__(256) k_pcg_direction(int64_t n, int it, int maxit, double tol2,
                                                       const double* __restrict__ r, const double* __restrict__ Minv,
                                                       double* __restrict__ p, const double* __restrict__ scal,
                                                       PcgFlags* __restrict__ flags) {
    if (flags->done) return;
    const bool first = blockIdx.x == 0 && threadIdx.x == 0;
    if (flags->breakdown) { if (first) flags->done = 1; return; }
    const bool dev_it = it < 0;
    if (dev_it) it = flags->it;
    const double rr = scal[4 * it + 1];
    const bool stop = rr <= tol2 * scal[1] || it >= maxit;
    if (first) { flags->iters = it; if (stop) flags->done = 1; }
    if (stop) return;
    const double beta = scal[4 * it + 2] / scal[4 * (it - 1) + 2];
    const int64_t n2 = n >> 1;
    const double2* r2 = reinterpret_cast<const double2*>(r);
    const double2* m2 = reinterpret_cast<const double2*>(Minv);
    double2* p2 = reinterpret_cast<double2*>(p);
    for (int64_t v = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; v < n2; v += (int64_t)gridDim.x * blockDim.x) {
        const double2 rv = r2[v], mv = m2[v];
        double2 pv = p2[v];
        pv.x = mv.x * rv.x + beta * pv.x;
        pv.y = mv.y * rv.y + beta * pv.y;
        p2[v] = pv;
    }
    if ((n & 1) && first) p[n - 1] = Minv[n - 1] * r[n - 1] + beta * p[n - 1];
    if (dev_it) {                                       // the last block to finish advances the iteration, clears p.q
        __shared__ unsigned int last;
        __syncthreads();
        if (threadIdx.x == 0) last = atomicAdd(&flags->ticket, 1u) == gridDim.x - 1;
        __syncthreads();
        if (last && threadIdx.x == 0) { flags->ticket = 0; flags->pq = 0.0; flags->it = it + 1; }
    }
}

}  // namespace

extern "C" int sem_pcg(sem_ctx* c, const double* b, double* x, double tol, int maxit, int* iters_out,
                       double* relres_out) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (!b || !x) return sem_fail(c, SEM_EINVAL, "sem_pcg: NULL vector");
    if (((uintptr_t)x % 16) || ((uintptr_t)b % 8)) return sem_fail(c, SEM_EINVAL, "sem_pcg: x must be 16-byte aligned");
    if (!(tol > 0.0) && maxit <= 0) return sem_fail(c, SEM_EINVAL, "sem_pcg: tol <= 0 with maxit <= 0");
    if (!c->geom_done) return sem_fail(c, SEM_ESTATE, "sem_pcg before sem_geom");
    if (c->lambda != 0.0 && !c->with_mass) return sem_fail(c, SEM_ESTATE, "lambda != 0 needs with_mass");
    if (maxit < 0) maxit = 0;
    if (c->inner) return sem_inner_pcg(c, b, x, tol, maxit, iters_out, relres_out);     // sem_inner.cu
    cudaStream_t st = c->stream;
    const int64_t n = c->nL;
    if (!c->pcg_ready || c->lambda_of_diag != c->lambda) {
        int rc = sem_build_diag(c);
        if (rc) return rc;
        if (!c->d_r) {
            SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_r, n * sizeof(double)));
            SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_p, n * sizeof(double)));
            SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_w, n * sizeof(double)));
        }
        c->pcg_ready = true;
    }
    const int64_t need = 4 * ((int64_t)maxit + 2) + 8;      // doubles; the flags (40 bytes) live after the slots
    if (need > c->scal_cap) {
        cudaFree(c->d_scal);
        c->d_scal = nullptr;
        SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_scal, need * sizeof(double)));
        c->scal_cap = need;
    }
    double* scal = c->d_scal;
    PcgFlags* flags = reinterpret_cast<PcgFlags*>(scal + 4 * ((int64_t)maxit + 2));
    SEM_CUDA_OK(c, cudaMemsetAsync(scal, 0, need * sizeof(double), st));
    const unsigned vgrid = (unsigned)c->num_sms * 8;

    // r = M b - A (M x0)
    k_mask_vec<<<vgrid, 256, 0, st>>>(n, c->d_wt, x);
    int rc = sem_launch_ax_gs(c, x, c->d_w, SEM_F64, c->lambda, nullptr, nullptr);
    if (rc) return rc;
    k_pcg_init<<<vgrid, 256, 0, st>>>(n, b, c->d_w, c->d_Minv, c->d_wt, x, c->d_r, c->d_p, scal);
    double h0[4];
    SEM_CUDA_OK(c, cudaMemcpyAsync(h0, scal, 4 * sizeof(double), cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    SEM_CUDA_OK(c, cudaGetLastError());
    const double rr0 = h0[1];
    int iters = 0;
    PcgFlags hf = {};
    if (rr0 > 0.0 && maxit > 0) {
        const double tol2 = tol > 0.0 ? tol * tol : 0.0;
        const int batch = 16;
        auto iteration = [&](int it) -> int {            // it < 0: iteration number and p.q on the device (graph replay)
            double* dot = it < 0 ? &flags->pq : scal + 4 * it;
            int r1 = sem_launch_ax_gs(c, c->d_p, c->d_w, SEM_F64, c->lambda, dot, &flags->done);
            if (r1) return r1;
            if (c->d_wt8)
                k_pcg_update<true><<<vgrid, 256, 0, st>>>(n, it, c->d_p, c->d_w, c->d_Minv, c->d_wt, c->d_wt8, x, c->d_r, scal, flags);
            else
                k_pcg_update<false><<<vgrid, 256, 0, st>>>(n, it, c->d_p, c->d_w, c->d_Minv, c->d_wt, nullptr, x, c->d_r, scal, flags);
            k_pcg_direction<<<vgrid, 256, 0, st>>>(n, it, maxit, tol2, c->d_r, c->d_Minv, c->d_p, scal, flags);
            return SEM_OK;
        };
        // One CUDA graph of `batch` iterations, replayed until the device raises `done` (non-default streams; meshes
        // whose operator is a single launch pair).  The kernels' sum is what an iteration costs; the ~2 us of stream-launch
        // gap per kernel is what the graph removes.
        cudaGraphExec_t gexec = nullptr;
        const bool graphable = st != nullptr && st != cudaStreamLegacy && c->chunk_e0.size() < 3 && maxit >= batch;
        if (graphable && cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            for (int q = 0; q < batch && rc == SEM_OK; ++q) rc = iteration(-1);
            cudaGraph_t graph = nullptr;
            const cudaError_t e = cudaStreamEndCapture(st, &graph);
            if (rc != SEM_OK || e != cudaSuccess || !graph || cudaGraphInstantiate(&gexec, graph, 0) != cudaSuccess) gexec = nullptr;
            if (graph) cudaGraphDestroy(graph);
            cudaGetLastError();
            if (rc != SEM_OK) return rc;
        } else {
            cudaGetLastError();
        }
        if (gexec) {
            const int one = 1;
            SEM_CUDA_OK(c, cudaMemcpyAsync(&flags->it, &one, sizeof(int), cudaMemcpyHostToDevice, st));
            for (int it0 = 1; it0 <= maxit; it0 += batch) {
                SEM_CUDA_OK(c, cudaGraphLaunch(gexec, st));
                SEM_CUDA_OK(c, cudaMemcpyAsync(&hf, flags, sizeof(hf), cudaMemcpyDeviceToHost, st));
                SEM_CUDA_OK(c, cudaStreamSynchronize(st));
                if (hf.done) break;
            }
            cudaGraphExecDestroy(gexec);
        } else {
            for (int it = 1; it <= maxit; ++it) {
                if ((rc = iteration(it))) return rc;
                if (it % batch == 0 || it == maxit) {
                    SEM_CUDA_OK(c, cudaMemcpyAsync(&hf, flags, sizeof(hf), cudaMemcpyDeviceToHost, st));
                    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
                    if (hf.done) break;
                }
            }
        }
        SEM_CUDA_OK(c, cudaGetLastError());
        iters = hf.iters;
    }
    // residual history from the per-iteration slots
    delete[] c->h_hist;
    c->h_hist = new double[iters + 1];
    c->hist_n = iters + 1;
    c->h_hist[0] = rr0 > 0.0 ? 1.0 : 0.0;
    if (iters > 0) {
        double* slots = new double[4 * ((size_t)iters + 1)];
        cudaError_t e = cudaMemcpyAsync(slots, scal, 4 * ((size_t)iters + 1) * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { delete[] slots; return sem_fail(c, SEM_ECUDA, "pcg history: %s", cudaGetErrorString(e)); }
        for (int i = 1; i <= iters; ++i) c->h_hist[i] = sqrt(slots[4 * i + 1] / rr0);
        if (hf.breakdown) c->h_hist[iters] = c->h_hist[iters - 1];    // the failed iteration did not update r
        delete[] slots;
    }
    if (iters_out) *iters_out = iters;
    if (relres_out) *relres_out = c->h_hist[iters];
    return SEM_OK;
}


// ---------------------------------------------------------------------------------------------------------------
// NEXT-4: the same recurrence with the elements partitioned over ranks.  Each rank runs this call on
// its own context with its part of b and x.  Per iteration: the sharded operator (sem_shard.cu: rank-local operator and
// gather-scatter, interface exchange through the hooks, started after the interface chunk when sem_shard_set_interface
// was called), ONE all-reduce of p.q, the update kernel, ONE all-reduce of (r.r, r.z), the direction kernel.  The
// scalars stay on the device as in sem_pcg: the all-reduce works in place on the iteration's slot, every rank then
// holds the same bits, takes the same stopping decision, and the host polls the flag every 8 iterations.  Dot weights
// are 1 / (multiplicity over ALL ranks), the preconditioner is the diagonal assembled over all ranks.
// ---------------------------------------------------------------------------------------------------------------
extern "C" int sem_pcg_sharded(sem_ctx* c, const double* b, double* x, double tol, int maxit,
                               const sem_shard_hooks* hooks, int* iters_out, double* relres_out) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (!b || !x) return sem_fail(c, SEM_EINVAL, "sem_pcg_sharded: NULL vector");
    if (((uintptr_t)x % 16) || ((uintptr_t)b % 8)) return sem_fail(c, SEM_EINVAL, "sem_pcg_sharded: x must be 16-byte aligned");
    if (!(tol > 0.0) && maxit <= 0) return sem_fail(c, SEM_EINVAL, "sem_pcg_sharded: tol <= 0 with maxit <= 0");
    if (!c->geom_done) return sem_fail(c, SEM_ESTATE, "sem_pcg_sharded before sem_geom");
    if (c->lambda != 0.0 && !c->with_mass) return sem_fail(c, SEM_ESTATE, "lambda != 0 needs with_mass");
    int rc = sem_hooks_ok(c, hooks, "sem_pcg_sharded");
    if (rc) return rc;
    if (maxit < 0) maxit = 0;
    cudaStream_t st = c->stream;
    const int64_t n = c->nL;
    if (!c->d_Minv_g || c->lambda_of_shard != c->lambda)
        if ((rc = sem_shard_build_diag(c, hooks))) return rc;
    if (!c->d_r) {
        SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_r, n * sizeof(double)));
        SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_p, n * sizeof(double)));
        SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_w, n * sizeof(double)));
    }
    const int64_t need = 4 * ((int64_t)maxit + 2) + 8;
    if (need > c->scal_cap) {
        cudaFree(c->d_scal);
        c->d_scal = nullptr;
        SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_scal, need * sizeof(double)));
        c->scal_cap = need;
    }
    double* scal = c->d_scal;
    PcgFlags* flags = reinterpret_cast<PcgFlags*>(scal + 4 * ((int64_t)maxit + 2));
    SEM_CUDA_OK(c, cudaMemsetAsync(scal, 0, need * sizeof(double), st));
    const unsigned vgrid = (unsigned)c->num_sms * 8;
    auto reduce = [&](double* p, int cnt) -> int {
        return hooks->allreduce(hooks->user, p, cnt) ? sem_fail(c, SEM_ECUDA, "sem_pcg_sharded: allreduce hook failed") : SEM_OK;
    };

    k_mask_vec<<<vgrid, 256, 0, st>>>(n, c->d_wt_g, x);
    if ((rc = sem_launch_ax_gs_sharded(c, x, c->d_w, SEM_F64, c->lambda, nullptr, nullptr, hooks))) return rc;
    k_pcg_init<<<vgrid, 256, 0, st>>>(n, b, c->d_w, c->d_Minv_g, c->d_wt_g, x, c->d_r, c->d_p, scal);
    if ((rc = reduce(scal + 1, 2))) return rc;
    double h0[4];
    SEM_CUDA_OK(c, cudaMemcpyAsync(h0, scal, 4 * sizeof(double), cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    SEM_CUDA_OK(c, cudaGetLastError());
    const double rr0 = h0[1];
    int iters = 0;
    PcgFlags hf = {};
    if (rr0 > 0.0 && maxit > 0) {
        const double tol2 = tol > 0.0 ? tol * tol : 0.0;
        const int batch = 8;
        for (int it = 1; it <= maxit; ++it) {
            if ((rc = sem_launch_ax_gs_sharded(c, c->d_p, c->d_w, SEM_F64, c->lambda, scal + 4 * it, &flags->done, hooks))) return rc;
            if ((rc = reduce(scal + 4 * it, 1))) return rc;
            k_pcg_update<false><<<vgrid, 256, 0, st>>>(n, it, c->d_p, c->d_w, c->d_Minv_g, c->d_wt_g, nullptr, x, c->d_r, scal, flags);
            if ((rc = reduce(scal + 4 * it + 1, 2))) return rc;
            k_pcg_direction<<<vgrid, 256, 0, st>>>(n, it, maxit, tol2, c->d_r, c->d_Minv_g, c->d_p, scal, flags);
            if (it % batch == 0 || it == maxit) {
                SEM_CUDA_OK(c, cudaMemcpyAsync(&hf, flags, sizeof(hf), cudaMemcpyDeviceToHost, st));
                SEM_CUDA_OK(c, cudaStreamSynchronize(st));
                if (hf.done) break;
            }
        }
        SEM_CUDA_OK(c, cudaGetLastError());
        iters = hf.iters;
    }
    delete[] c->h_hist;
    c->h_hist = new double[iters + 1];
    c->hist_n = iters + 1;
    c->h_hist[0] = rr0 > 0.0 ? 1.0 : 0.0;
    if (iters > 0) {
        double* slots = new double[4 * ((size_t)iters + 1)];
        cudaError_t e = cudaMemcpyAsync(slots, scal, 4 * ((size_t)iters + 1) * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { delete[] slots; return sem_fail(c, SEM_ECUDA, "pcg history: %s", cudaGetErrorString(e)); }
        for (int i = 1; i <= iters; ++i) c->h_hist[i] = sqrt(slots[4 * i + 1] / rr0);
        if (hf.breakdown) c->h_hist[iters] = c->h_hist[iters - 1];
        delete[] slots;
    }
    if (iters_out) *iters_out = iters;
    if (relres_out) *relres_out = c->h_hist[iters];
    return SEM_OK;
}


// ---------------------------------------------------------------------------------------------------------------
// NEXT-4: Jacobi-PCG on nf right-hand sides at once ("3 Helmholtz problems -- one for each velocity component ...
// Jacobi-preconditioned conjugate gradient iteration").  Every field runs exactly the recurrence of sem_pcg with its own
// alpha, beta, stopping test and breakdown flag (own scalar slots), so each field's iterates are those sem_pcg would
// produce for it alone; what is shared is the operator pass: one sem_launch_ax_many reads G once for all fields, and
// one gather-scatter launch handles up to 4 of them.  The loop ends when every field has stopped.
// ---------------------------------------------------------------------------------------------------------------
namespace {
__global__ void k_all_done(int nf, const PcgFlags* const* flags, int* __restrict__ all_done) {
    int d = 1;
    for (int f = 0; f < nf; ++f) d &= flags[f]->done != 0;
    *all_done = d;
}

// The two vector kernels of an iteration for NF fields at once (field f at + f * fs): exactly k_pcg_update /
// k_pcg_direction per field (own alpha, beta, flags, slots), but Minv and the dot weights are read once for all fields
// (57 -> 48 + 9 / NF and 32 -> 24 + 8 / NF bytes per node and field).
template <int NF>
struct ManyArgs {
    double* scal[NF];
    PcgFlags* flags[NF];
};

template <bool W8, int NF>
__global__ void __launch_bounds__(256) k_pcg_update_many(int64_t n, int it_arg, const double* __restrict__ p,
                                                         const double* __restrict__ w, const double* __restrict__ Minv,
                                                         const double* __restrict__ wt, const uint8_t* __restrict__ wt8,
                                                         double* __restrict__ x, double* __restrict__ r, int64_t fs,
                                                         ManyArgs<NF> a) {
    bool act[NF];
    double alpha[NF];
    int itf[NF];
    bool any = false;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
        PcgFlags* fl = a.flags[f];
        act[f] = false; alpha[f] = 0.0; itf[f] = 0;
        if (fl->done) continue;
        const bool dev_it = it_arg < 0;
        const int it = dev_it ? fl->it : it_arg;
        const double pq = dev_it ? fl->pq : a.scal[f][4 * it + 0];
        if (dev_it && blockIdx.x == 0 && threadIdx.x == 0) a.scal[f][4 * it + 0] = pq;
        if (!(pq > 0.0)) {                              // breakdown (S13): stop this field, keep its x
            if (blockIdx.x == 0 && threadIdx.x == 0) { fl->breakdown = 1; fl->iters = it; }
            continue;
        }
        act[f] = true; any = true; itf[f] = it;
        alpha[f] = a.scal[f][4 * (it - 1) + 2] / pq;
    }
    if (!any) return;
    double srr[NF], srz[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) { srr[f] = 0.0; srz[f] = 0.0; }
    const int64_t n2 = n >> 1;
    const double2* m2 = reinterpret_cast<const double2*>(Minv);
    const double2* t2 = reinterpret_cast<const double2*>(wt);
    for (int64_t v = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; v < n2; v += (int64_t)gridDim.x * blockDim.x) {
        const double2 mv = m2[v];
        double2 tv;
        if constexpr (W8) {
            const uchar2 c8 = reinterpret_cast<const uchar2*>(wt8)[v];
            tv = make_double2(wt_of(c8.x), wt_of(c8.y));
        } else {
            tv = t2[v];
        }
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            if (!act[f]) continue;
            const double2 pv = reinterpret_cast<const double2*>(p + f * fs)[v], wv = reinterpret_cast<const double2*>(w + f * fs)[v];
            double2 xv = reinterpret_cast<double2*>(x + f * fs)[v], rv = reinterpret_cast<double2*>(r + f * fs)[v];
            xv.x += alpha[f] * pv.x; xv.y += alpha[f] * pv.y;
            rv.x -= alpha[f] * wv.x; rv.y -= alpha[f] * wv.y;
            reinterpret_cast<double2*>(x + f * fs)[v] = xv;
            reinterpret_cast<double2*>(r + f * fs)[v] = rv;
            const double ax = tv.x * rv.x * rv.x, ay = tv.y * rv.y * rv.y;
            srr[f] += ax + ay;
            srz[f] += ax * mv.x + ay * mv.y;
        }
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const int64_t l = n - 1;
        const double wl = W8 ? wt_of(wt8[l]) : wt[l];
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            if (!act[f]) continue;
            x[f * fs + l] += alpha[f] * p[f * fs + l];
            const double rl = r[f * fs + l] - alpha[f] * w[f * fs + l];
            r[f * fs + l] = rl;
            srr[f] += wl * rl * rl;
            srz[f] += wl * rl * rl * Minv[l];
        }
    }
#pragma unroll
    for (int f = 0; f < NF; ++f) {
        if (act[f]) block_sum2_atomic(srr[f], srz[f], a.scal[f] + 4 * itf[f] + 1, a.scal[f] + 4 * itf[f] + 2);
        __syncthreads();                                // the reduction's shared buffer is reused by the next field
    }
}

template <int NF>
__global__ void __launch_bounds__(256) k_pcg_direction_many(int64_t n, int it_arg, int maxit, double tol2,
                                                            const double* __restrict__ r, const double* __restrict__ Minv,
                                                            double* __restrict__ p, int64_t fs, ManyArgs<NF> a) {
    const bool first = blockIdx.x == 0 && threadIdx.x == 0;
    const bool dev_it = it_arg < 0;
    bool act[NF];
    double beta[NF];
    int itf[NF];
    bool any = false;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
        PcgFlags* fl = a.flags[f];
        act[f] = false; beta[f] = 0.0; itf[f] = 0;
        if (fl->done) continue;
        if (fl->breakdown) { if (first) fl->done = 1; continue; }
        const int it = dev_it ? fl->it : it_arg;
        const double rr = a.scal[f][4 * it + 1];
        const bool stop = rr <= tol2 * a.scal[f][1] || it >= maxit;
        if (first) { fl->iters = it; if (stop) fl->done = 1; }
        if (stop) continue;
        act[f] = true; any = true; itf[f] = it;
        beta[f] = a.scal[f][4 * it + 2] / a.scal[f][4 * (it - 1) + 2];
    }
    if (!any) return;
    const int64_t n2 = n >> 1;
    const double2* m2 = reinterpret_cast<const double2*>(Minv);
    for (int64_t v = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; v < n2; v += (int64_t)gridDim.x * blockDim.x) {
        const double2 mv = m2[v];
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            if (!act[f]) continue;
            const double2 rv = reinterpret_cast<const double2*>(r + f * fs)[v];
            double2 pv = reinterpret_cast<double2*>(p + f * fs)[v];
            pv.x = mv.x * rv.x + beta[f] * pv.x;
            pv.y = mv.y * rv.y + beta[f] * pv.y;
            reinterpret_cast<double2*>(p + f * fs)[v] = pv;
        }
    }
    if ((n & 1) && first) {
#pragma unroll
        for (int f = 0; f < NF; ++f)
            if (act[f]) p[f * fs + n - 1] = Minv[n - 1] * r[f * fs + n - 1] + beta[f] * p[f * fs + n - 1];
    }
    if (dev_it) {                                       // per field: the last block advances the iteration, clears p.q
        __shared__ unsigned int last[NF];
        __syncthreads();
        if (threadIdx.x == 0) {
#pragma unroll
            for (int f = 0; f < NF; ++f) last[f] = act[f] ? (atomicAdd(&a.flags[f]->ticket, 1u) == gridDim.x - 1) : 0u;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
#pragma unroll
            for (int f = 0; f < NF; ++f)
                if (last[f]) { a.flags[f]->ticket = 0; a.flags[f]->pq = 0.0; a.flags[f]->it = itf[f] + 1; }
        }
    }
}
}  // namespace

extern "C" int sem_pcg_many(sem_ctx* c, const double* b, double* x, int nfields, int64_t field_stride, double tol,
                            int maxit, int* iters_out, double* relres_out) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (!b || !x) return sem_fail(c, SEM_EINVAL, "sem_pcg_many: NULL vector");
    if (nfields < 1 || nfields > 8 || field_stride < c->nL || (field_stride & 1))
        return sem_fail(c, SEM_EINVAL, "sem_pcg_many: need 1 <= nfields <= 8 and an even field_stride >= nL");
    if (((uintptr_t)x % 16) || ((uintptr_t)b % 8)) return sem_fail(c, SEM_EINVAL, "sem_pcg_many: x must be 16-byte aligned");
    if (!(tol > 0.0) && maxit <= 0) return sem_fail(c, SEM_EINVAL, "sem_pcg_many: tol <= 0 with maxit <= 0");
    if (!c->geom_done) return sem_fail(c, SEM_ESTATE, "sem_pcg_many before sem_geom");
    if (c->lambda != 0.0 && !c->with_mass) return sem_fail(c, SEM_ESTATE, "lambda != 0 needs with_mass");
    if (maxit < 0) maxit = 0;
    cudaStream_t st = c->stream;
    const int64_t n = c->nL, fs = field_stride;
    const int nf = nfields;
    int rc;
    if (!c->pcg_ready || c->lambda_of_diag != c->lambda) {
        if ((rc = sem_build_diag(c))) return rc;
        if (!c->d_r) {
            SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_r, n * sizeof(double)));
            SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_p, n * sizeof(double)));
            SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_w, n * sizeof(double)));
        }
        c->pcg_ready = true;
    }
    // work vectors r, p, w of all fields at the caller's stride; per-field scalar slots and flags
    const int64_t slot = 4 * ((int64_t)maxit + 2) + 8;           // doubles per field (as in sem_pcg)
    double *R = nullptr, *P = nullptr, *W = nullptr, *scal = nullptr;
    const PcgFlags** d_fl = nullptr;
    int* d_all = nullptr;
    auto cleanup = [&]() { cudaFree(R); cudaFree(P); cudaFree(W); cudaFree(scal); cudaFree((void*)d_fl); cudaFree(d_all); };
    cudaError_t e = cudaMalloc((void**)&R, nf * fs * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&P, nf * fs * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&W, nf * fs * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&scal, nf * slot * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&d_fl, nf * sizeof(PcgFlags*));
    if (e == cudaSuccess) e = cudaMalloc((void**)&d_all, sizeof(int));
    if (e != cudaSuccess) { cleanup(); return sem_fail(c, SEM_ENOMEM, "sem_pcg_many: %s", cudaGetErrorString(e)); }
    auto fail = [&](int code) { cudaStreamSynchronize(st); cleanup(); return code; };
    PcgFlags* fl[8];
    for (int f = 0; f < nf; ++f) fl[f] = reinterpret_cast<PcgFlags*>(scal + f * slot + 4 * ((int64_t)maxit + 2));
    cudaMemsetAsync(scal, 0, nf * slot * sizeof(double), st);
    cudaMemsetAsync(d_all, 0, sizeof(int), st);
    cudaMemcpyAsync((void*)d_fl, fl, nf * sizeof(PcgFlags*), cudaMemcpyHostToDevice, st);
    const unsigned vgrid = (unsigned)c->num_sms * 8;
    for (int f = 0; f < nf; ++f) k_mask_vec<<<vgrid, 256, 0, st>>>(n, c->d_wt, x + f * fs);
    if ((rc = sem_launch_ax_many(c, x, W, nf, fs, SEM_F64, c->lambda, nullptr, 0, nullptr))) return fail(rc);
    if ((rc = sem_launch_gs_fields(c, W, nf, fs, SEM_F64, true, nullptr))) return fail(rc);
    for (int f = 0; f < nf; ++f)
        k_pcg_init<<<vgrid, 256, 0, st>>>(n, b + f * fs, W + f * fs, c->d_Minv, c->d_wt, x + f * fs, R + f * fs, P + f * fs,
                                          scal + f * slot);
    double rr0[8];
    for (int f = 0; f < nf; ++f) {
        double h0[4];
        cudaMemcpyAsync(h0, scal + f * slot, 4 * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (cudaStreamSynchronize(st) != cudaSuccess) return fail(sem_fail(c, SEM_ECUDA, "sem_pcg_many: init failed"));
        rr0[f] = h0[1];
    }
    const double tol2 = tol > 0.0 ? tol * tol : 0.0;
    // a field with a zero initial residual has nothing to do: raise its flag now
    for (int f = 0; f < nf; ++f)
        if (!(rr0[f] > 0.0) || maxit == 0) {
            PcgFlags done = {};
            done.done = 1;
            cudaMemcpyAsync(fl[f], &done, sizeof(done), cudaMemcpyHostToDevice, st);
        }
    PcgFlags hf[8] = {};
    const int batch = 16;
    auto iteration = [&](int it) -> int {                // it < 0: iteration numbers and p.q on the device (graph replay)
        k_all_done<<<1, 1, 0, st>>>(nf, d_fl, d_all);
        double* dot = it < 0 ? &fl[0]->pq : scal + 4 * it;      // field f: + f * slot doubles in both cases
        int r1 = sem_launch_ax_many(c, P, W, nf, fs, SEM_F64, c->lambda, dot, slot, d_all);
        if (r1) return r1;
        if ((r1 = sem_launch_gs_fields(c, W, nf, fs, SEM_F64, true, d_all))) return r1;
        for (int f = 0; f < nf;) {                           // groups of 3 or 2 fields share Minv and the dot weights
            const int left = nf - f, take = left >= 3 && left != 4 ? 3 : (left >= 2 ? 2 : 1);
            double* sc = scal + f * slot;
            if (take == 3) {
                ManyArgs<3> a = {{sc, sc + slot, sc + 2 * slot}, {fl[f], fl[f + 1], fl[f + 2]}};
                if (c->d_wt8) k_pcg_update_many<true, 3><<<vgrid, 256, 0, st>>>(n, it, P + f * fs, W + f * fs, c->d_Minv, c->d_wt, c->d_wt8, x + f * fs, R + f * fs, fs, a);
                else k_pcg_update_many<false, 3><<<vgrid, 256, 0, st>>>(n, it, P + f * fs, W + f * fs, c->d_Minv, c->d_wt, nullptr, x + f * fs, R + f * fs, fs, a);
                k_pcg_direction_many<3><<<vgrid, 256, 0, st>>>(n, it, maxit, tol2, R + f * fs, c->d_Minv, P + f * fs, fs, a);
            } else if (take == 2) {
                ManyArgs<2> a = {{sc, sc + slot}, {fl[f], fl[f + 1]}};
                if (c->d_wt8) k_pcg_update_many<true, 2><<<vgrid, 256, 0, st>>>(n, it, P + f * fs, W + f * fs, c->d_Minv, c->d_wt, c->d_wt8, x + f * fs, R + f * fs, fs, a);
                else k_pcg_update_many<false, 2><<<vgrid, 256, 0, st>>>(n, it, P + f * fs, W + f * fs, c->d_Minv, c->d_wt, nullptr, x + f * fs, R + f * fs, fs, a);
                k_pcg_direction_many<2><<<vgrid, 256, 0, st>>>(n, it, maxit, tol2, R + f * fs, c->d_Minv, P + f * fs, fs, a);
            } else {
                if (c->d_wt8)
                    k_pcg_update<true><<<vgrid, 256, 0, st>>>(n, it, P + f * fs, W + f * fs, c->d_Minv, c->d_wt, c->d_wt8, x + f * fs, R + f * fs, sc, fl[f]);
                else
                    k_pcg_update<false><<<vgrid, 256, 0, st>>>(n, it, P + f * fs, W + f * fs, c->d_Minv, c->d_wt, nullptr, x + f * fs, R + f * fs, sc, fl[f]);
                k_pcg_direction<<<vgrid, 256, 0, st>>>(n, it, maxit, tol2, R + f * fs, c->d_Minv, P + f * fs, sc, fl[f]);
            }
            f += take;
        }
        return SEM_OK;
    };
    auto poll = [&](bool& all) -> int {
        all = true;
        for (int f = 0; f < nf; ++f) cudaMemcpyAsync(&hf[f], fl[f], sizeof(PcgFlags), cudaMemcpyDeviceToHost, st);
        if (cudaStreamSynchronize(st) != cudaSuccess) return sem_fail(c, SEM_ECUDA, "sem_pcg_many: loop failed");
        for (int f = 0; f < nf; ++f) all = all && hf[f].done;
        return SEM_OK;
    };
    // as in sem_pcg: one CUDA graph of `batch` lockstep iterations, replayed until every field has stopped
    cudaGraphExec_t gexec = nullptr;
    const bool graphable = st != nullptr && st != cudaStreamLegacy && maxit >= batch;
    if (graphable && cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
        rc = SEM_OK;
        for (int q = 0; q < batch && rc == SEM_OK; ++q) rc = iteration(-1);
        cudaGraph_t graph = nullptr;
        const cudaError_t ec = cudaStreamEndCapture(st, &graph);
        if (rc != SEM_OK || ec != cudaSuccess || !graph || cudaGraphInstantiate(&gexec, graph, 0) != cudaSuccess) gexec = nullptr;
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        if (rc != SEM_OK) return fail(rc);
    } else {
        cudaGetLastError();
    }
    if (gexec) {
        const int one = 1;
        for (int f = 0; f < nf; ++f) cudaMemcpyAsync(&fl[f]->it, &one, sizeof(int), cudaMemcpyHostToDevice, st);
        for (int it0 = 1; it0 <= maxit; it0 += batch) {
            bool all = false;
            if (cudaGraphLaunch(gexec, st) != cudaSuccess || (rc = poll(all))) {
                cudaGraphExecDestroy(gexec);
                return fail(rc ? rc : sem_fail(c, SEM_ECUDA, "sem_pcg_many: graph launch failed"));
            }
            if (all) break;
        }
        cudaGraphExecDestroy(gexec);
    } else {
        for (int it = 1; it <= maxit; ++it) {
            if ((rc = iteration(it))) return fail(rc);
            if (it % batch == 0 || it == maxit) {
                bool all = false;
                if ((rc = poll(all))) return fail(rc);
                if (all) break;
            }
        }
    }
    if (cudaGetLastError() != cudaSuccess) return fail(sem_fail(c, SEM_ECUDA, "sem_pcg_many: launch failed"));
    for (int f = 0; f < nf; ++f) {
        const int iters = hf[f].iters;
        double rel = rr0[f] > 0.0 ? 1.0 : 0.0;
        if (iters > 0) {
            double s1[4], s0[4];
            cudaMemcpyAsync(s1, scal + f * slot + 4 * (int64_t)iters, sizeof(s1), cudaMemcpyDeviceToHost, st);
            cudaMemcpyAsync(s0, scal + f * slot + 4 * (int64_t)(iters - 1), sizeof(s0), cudaMemcpyDeviceToHost, st);
            cudaStreamSynchronize(st);
            rel = hf[f].breakdown ? (iters > 1 ? sqrt(s0[1] / rr0[f]) : 1.0) : sqrt(s1[1] / rr0[f]);
        }
        if (iters_out) iters_out[f] = iters;
        if (relres_out) relres_out[f] = rel;
    }
    cudaStreamSynchronize(st);
    cleanup();
    return SEM_OK;
}
