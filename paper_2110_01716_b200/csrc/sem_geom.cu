// sem_geom.cu — a2 (setup): geometric factors, the exact Jacobi diagonal, and the layout conversions around them.
// P:69 (isoparametric map), O3 (G, B, detJ), O7 (exact diagonal incl. cross terms), S16 (FP32 copy rounded once).
//
// Device layout of G ("slab layout", library-owned): Gs[grp][k][slot][c][j*p+i], grp = e / epb, slot = e % epb,
// c = rr,rs,rt,ss,st,tt (sem_g_off in sem_internal.h), so that the six factors of one k-slab of one element group
// are one contiguous chunk (one bulk copy in the Ax kernel).  The array is padded with zeros to whole groups.
#include "sem_geom_dev.cuh"
#include "sem_internal.h"

namespace {

inline unsigned nblk(int64_t n, int t = 256) { return (unsigned)((n + t - 1) / t); }

// One thread per node.  xyz == nullptr: analytic trilinear Jacobian (S5); else D applied to xyz (isoparametric).
__global__ void k_geom(int64_t E, int p, int epb, Gll1D gll, const double* __restrict__ vert,
                       const double* __restrict__ xyz, int64_t slab, double* __restrict__ Gs, double* __restrict__ Bm, double* __restrict__ detJ,
                       int* __restrict__ bad) {
    const int64_t p2 = (int64_t)p * p, p3 = p2 * p;
    const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (l >= E * p3) return;
    const int64_t e = l / p3;
    const int n = (int)(l - e * p3);
    const int k = n / (int)p2, j = (n / p) % p, i = n % p;
    double J[3][3];
    if (xyz == nullptr) {
        double X[8][3], cf[8][3];
#pragma unroll
        for (int v = 0; v < 8; ++v)
#pragma unroll
            for (int d = 0; d < 3; ++d) X[v][d] = vert[(e * 8 + v) * 3 + d];
        sem_trilinear_coef(X, cf);
        sem_trilinear_jac(cf, gll.xi[i], gll.xi[j], gll.xi[k], J);
    } else {
        const double* Xe = xyz + e * p3 * 3;
        for (int a = 0; a < 3; ++a) {
            double dr = 0, ds = 0, dt = 0;
            for (int m = 0; m < p; ++m) {
                dr += gll.D[i * p + m] * Xe[((int64_t)(k * p + j) * p + m) * 3 + a];
                ds += gll.D[j * p + m] * Xe[((int64_t)(k * p + m) * p + i) * 3 + a];
                dt += gll.D[k * p + m] * Xe[((int64_t)(m * p + j) * p + i) * 3 + a];
            }
            J[a][0] = dr; J[a][1] = ds; J[a][2] = dt;
        }
    }
    double g[6], B;
    const double det = sem_factors(J, gll.rho[i] * gll.rho[j] * gll.rho[k], g, B);
    if (!(det > 0.0)) atomicOr(bad, 1);
    double* slab_ptr = Gs + sem_g_off(e, k, p, epb, slab) + (j * p + i);
#pragma unroll
    for (int c = 0; c < 6; ++c) slab_ptr[c * p2] = g[c];
    if (Bm) Bm[l] = B;
    detJ[l] = det;
}

template <typename Tin, typename Tout>
__global__ void k_convert(int64_t n, const Tin* __restrict__ in, Tout* __restrict__ out) {
    int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (; t < n; t += stride) out[t] = (Tout)in[t];
}

// slab layout (stride slab_in) -> FP32 slab layout (stride slab_out)
__global__ void k_g32(int64_t nslabs, int cnt, int64_t slab_in, int64_t slab_out, const double* __restrict__ in,
                      float* __restrict__ out) {
    int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int64_t total = nslabs * cnt;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (; t < total; t += stride) {
        const int64_t s = t / cnt;
        const int r = (int)(t - s * cnt);
        out[s * slab_out + r] = (float)in[s * slab_in + r];
    }
}

// O7: exact local diagonal.  One thread per node.
__global__ void k_diag_local(int64_t E, int p, int epb, Gll1D gll, int64_t slab, const double* __restrict__ Gs,
                             const double* __restrict__ Bm, double lambda, double* __restrict__ diag) {
    const int64_t p2 = (int64_t)p * p, p3 = p2 * p;
    const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (l >= E * p3) return;
    const int64_t e = l / p3;
    const int n = (int)(l - e * p3);
    const int k = n / (int)p2, j = (n / p) % p, i = n % p;
    auto G = [&](int c, int kk, int jj, int ii) { return Gs[sem_g_off(e, kk, p, epb, slab) + c * p2 + jj * p + ii]; };
    double d = 0.0;
    for (int m = 0; m < p; ++m) {
        const double di = gll.D[m * p + i], dj = gll.D[m * p + j], dk = gll.D[m * p + k];
        d += di * di * G(0, k, j, m);
        d += dj * dj * G(3, k, m, i);
        d += dk * dk * G(5, m, j, i);
    }
    const double dii = gll.D[i * p + i], djj = gll.D[j * p + j], dkk = gll.D[k * p + k];
    d += 2.0 * (dii * djj * G(1, k, j, i) + dii * dkk * G(2, k, j, i) + djj * dkk * G(4, k, j, i));
    if (lambda != 0.0) d += lambda * Bm[l];
    diag[l] = d;
}

// Minv = mask / diag (S12, S14); wt = mask / mult (unique-node dot weights in local storage, O8)
__global__ void k_minv_wt(int64_t n, const double* __restrict__ diag, const int32_t* __restrict__ l2u,
                          const int32_t* __restrict__ mult, const uint8_t* __restrict__ mask_u,
                          double* __restrict__ Minv, double* __restrict__ wt, uint8_t* __restrict__ wt8,
                          int* __restrict__ big_mult) {
    const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (l >= n) return;
    const int32_t g = l2u[l];
    const bool masked = mask_u && mask_u[g];
    Minv[l] = masked ? 0.0 : 1.0 / diag[l];
    wt[l] = masked ? 0.0 : 1.0 / (double)mult[g];
    wt8[l] = masked ? 0 : (uint8_t)(mult[g] & 255);
    if (mult[g] > 255) *big_mult = 1;                 // benign race: every writer stores 1
}

// slab layout -> [E][ncomp][p^3] export (+ B as 7th)
__global__ void k_export(int64_t E, int p, int epb, int ncomp, int64_t slab, const double* __restrict__ Gs,
                         const double* __restrict__ Bm, double* __restrict__ out) {
    const int64_t p2 = (int64_t)p * p, p3 = p2 * p;
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t >= E * ncomp * p3) return;
    const int64_t e = t / (ncomp * p3);
    const int64_t r = t - e * ncomp * p3;
    const int c = (int)(r / p3);
    const int n = (int)(r - c * p3);
    const int k = n / (int)p2, ji = n % (int)p2;
    out[t] = c < 6 ? Gs[sem_g_off(e, k, p, epb, slab) + c * p2 + ji] : Bm[e * p3 + n];
}

Gll1D make_gll(const sem_ctx* c) {
    Gll1D g;
    for (int i = 0; i < 16; ++i) { g.xi[i] = i < c->p ? c->xi[i] : 0.0; g.rho[i] = i < c->p ? c->rho[i] : 0.0; }
    for (int i = 0; i < 256; ++i) g.D[i] = i < c->p * c->p ? c->D[i] : 0.0;
    return g;
}

}  // namespace

int sem_build_geom(sem_ctx* c, const double* node_xyz_host) {
    cudaStream_t st = c->stream;
    const int p = c->p;
    const int64_t p2 = (int64_t)p * p;
    c->slab_f64 = 6 * p2;                                   // 48 p^2 bytes: always a multiple of 16
    c->slab_f32 = 6 * p2 + ((6 * p2 * 4) % 16 ? 2 : 0);     // pad odd p to a multiple of 16 bytes
    const int64_t gcount = c->ngroups * c->epb * p * c->slab_f64;       // padded to whole groups
    cudaFree(c->d_G); cudaFree(c->d_B); cudaFree(c->d_detJ); cudaFree(c->d_G32); cudaFree(c->d_B32);
    c->d_G = nullptr; c->d_B = nullptr; c->d_detJ = nullptr; c->d_G32 = nullptr; c->d_B32 = nullptr;
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_G, gcount * sizeof(double)));
    if (c->ngroups * c->epb != c->E) SEM_CUDA_OK(c, cudaMemsetAsync(c->d_G, 0, gcount * sizeof(double), st));
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_detJ, c->nL * sizeof(double)));
    if (c->with_mass) SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_B, c->nL * sizeof(double)));
    double* d_xyz = nullptr;
    if (node_xyz_host) {
        SEM_CUDA_OK(c, cudaMalloc((void**)&d_xyz, c->nL * 3 * sizeof(double)));
        cudaError_t e = cudaMemcpyAsync(d_xyz, node_xyz_host, c->nL * 3 * sizeof(double), cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) { cudaFree(d_xyz); return sem_fail(c, SEM_ECUDA, "copy node_xyz: %s", cudaGetErrorString(e)); }
    }
    int* d_bad = nullptr;
    cudaError_t e = cudaMalloc((void**)&d_bad, sizeof(int));
    if (e != cudaSuccess) { cudaFree(d_xyz); return sem_fail(c, SEM_ENOMEM, "cudaMalloc: %s", cudaGetErrorString(e)); }
    cudaMemsetAsync(d_bad, 0, sizeof(int), st);
    k_geom<<<nblk(c->nL), 256, 0, st>>>(c->E, p, c->epb, make_gll(c), c->d_vert, d_xyz, c->slab_f64, c->d_G, c->d_B, c->d_detJ,
                                         d_bad);
    int h_bad = 0;
    cudaMemcpyAsync(&h_bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost, st);
    e = cudaStreamSynchronize(st);
    cudaFree(d_bad);
    cudaFree(d_xyz);
    if (e != cudaSuccess) return sem_fail(c, SEM_ECUDA, "geometry kernel: %s", cudaGetErrorString(e));
    SEM_CUDA_OK(c, cudaGetLastError());
    if (h_bad) return sem_fail(c, SEM_EMESH, "non-positive Jacobian determinant in at least one node");
    sem_release_G(c);                    // recompute mode keeps no stored G (48 B per node): rebuilt on demand
    return SEM_OK;
}

// Recompute mode (a9): the operator never reads the stored G, so it is not kept; the Jacobi diagonal and sem_get_geom
// rebuild it from the vertices for the duration of the call (trilinear geometry only: sem_geom enforces it).
int sem_ensure_G(sem_ctx* c) {
    if (c->d_G) return SEM_OK;
    cudaStream_t st = c->stream;
    const int64_t gcount = c->ngroups * c->epb * c->p * c->slab_f64;
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_G, gcount * sizeof(double)));
    if (c->ngroups * c->epb != c->E) SEM_CUDA_OK(c, cudaMemsetAsync(c->d_G, 0, gcount * sizeof(double), st));
    int* d_bad = nullptr;
    SEM_CUDA_OK(c, cudaMalloc((void**)&d_bad, sizeof(int)));
    cudaMemsetAsync(d_bad, 0, sizeof(int), st);
    k_geom<<<nblk(c->nL), 256, 0, st>>>(c->E, c->p, c->epb, make_gll(c), c->d_vert, nullptr, c->slab_f64, c->d_G, c->d_B,
                                         c->d_detJ, d_bad);
    const cudaError_t e = cudaStreamSynchronize(st);
    cudaFree(d_bad);
    if (e != cudaSuccess) return sem_fail(c, SEM_ECUDA, "geometry kernel: %s", cudaGetErrorString(e));
    return SEM_OK;
}

void sem_release_G(sem_ctx* c) {
    if (c->gmode != SEM_G_RECOMPUTE || !c->d_G) return;
    cudaStreamSynchronize(c->stream);
    cudaFree(c->d_G);
    c->d_G = nullptr;
}

// FP32 copies (S16: rounded once from double): G32 in stored mode, B32 whenever the mass factor exists
int sem_build_g32(sem_ctx* c) {
    cudaStream_t st = c->stream;
    if (!c->d_G32 && c->gmode == SEM_G_STORED) {
        const int64_t nslabs = c->ngroups * c->epb * c->p;
        SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_G32, nslabs * c->slab_f32 * sizeof(float)));
        if (c->slab_f32 != c->slab_f64) SEM_CUDA_OK(c, cudaMemsetAsync(c->d_G32, 0, nslabs * c->slab_f32 * sizeof(float), st));
        k_g32<<<c->num_sms * 8, 256, 0, st>>>(nslabs, 6 * c->p * c->p, c->slab_f64, c->slab_f32, c->d_G, c->d_G32);
    }
    if (!c->d_B32 && c->with_mass) {
        SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_B32, c->nL * sizeof(float)));
        k_convert<double, float><<<c->num_sms * 8, 256, 0, st>>>(c->nL, c->d_B, c->d_B32);
    }
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

int sem_build_diag(sem_ctx* c) {
    cudaStream_t st = c->stream;
    if (!c->d_diag) {
        SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_diag, c->nL * sizeof(double)));
        SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_Minv, c->nL * sizeof(double)));
        SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_wt, c->nL * sizeof(double)));
    }
    int rc = sem_ensure_G(c);
    if (rc) return rc;
    k_diag_local<<<nblk(c->nL), 256, 0, st>>>(c->E, c->p, c->epb, make_gll(c), c->slab_f64, c->d_G, c->d_B, c->lambda, c->d_diag);
    sem_release_G(c);
    if ((rc = sem_launch_gs(c, c->d_diag, SEM_F64, /*apply_mask=*/false))) return rc;
    if (!c->d_wt8) SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_wt8, c->nL));
    int* d_big = nullptr;
    SEM_CUDA_OK(c, cudaMalloc((void**)&d_big, sizeof(int)));
    SEM_CUDA_OK(c, cudaMemsetAsync(d_big, 0, sizeof(int), st));
    k_minv_wt<<<nblk(c->nL), 256, 0, st>>>(c->nL, c->d_diag, c->d_l2u, c->d_mult, c->has_mask ? c->d_mask_u : nullptr,
                                            c->d_Minv, c->d_wt, c->d_wt8, d_big);
    int h_big = 0;
    cudaError_t eb = cudaMemcpyAsync(&h_big, d_big, sizeof(int), cudaMemcpyDeviceToHost, st);
    if (eb == cudaSuccess) eb = cudaStreamSynchronize(st);
    cudaFree(d_big);
    if (eb != cudaSuccess) return sem_fail(c, SEM_ECUDA, "diag: %s", cudaGetErrorString(eb));
    if (h_big) { cudaFree(c->d_wt8); c->d_wt8 = nullptr; }        // a multiplicity above 255: keep the 8-byte weights only
    SEM_CUDA_OK(c, cudaGetLastError());
    c->lambda_of_diag = c->lambda;
    c->lambda_of_minv32 = -1.0;       // the FP32 copy (sem_cheby.cu) is stale now
    return SEM_OK;
}

int sem_geom_export(sem_ctx* c, double* G_host, double* detJ_host) {
    cudaStream_t st = c->stream;
    if (G_host) {
        if (int rg = sem_ensure_G(c)) return rg;
        const int ncomp = c->with_mass ? 7 : 6;
        const int64_t cnt = c->E * ncomp * c->p3;
        double* d_out = nullptr;
        SEM_CUDA_OK(c, cudaMalloc((void**)&d_out, cnt * sizeof(double)));
        k_export<<<nblk(cnt), 256, 0, st>>>(c->E, c->p, c->epb, ncomp, c->slab_f64, c->d_G, c->d_B, d_out);
        cudaError_t e = cudaMemcpyAsync(G_host, d_out, cnt * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        cudaFree(d_out);
        sem_release_G(c);
        if (e != cudaSuccess) return sem_fail(c, SEM_ECUDA, "export G: %s", cudaGetErrorString(e));
    }
    if (detJ_host) {
        SEM_CUDA_OK(c, cudaMemcpyAsync(detJ_host, c->d_detJ, c->nL * sizeof(double), cudaMemcpyDeviceToHost, st));
        SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    }
    return SEM_OK;
}
