// sem_inner.cu — element renumbering for the solver's own vectors (BASELINE.json configs[4]: "element
// order randomly permuted (scrambled numbering to stress gather-scatter locality)").
// The caller's vectors live in the caller's element order and the C ABI keeps it.  But the Jacobi-PCG loop works on
// LIBRARY-owned vectors (r, p, w) and touches the caller's b and x once each, so for a large mesh whose element order has
// no locality the context keeps a second, inner context over the same elements sorted by their smallest global id (for
// the usual numberings that is a space-filling order; a lexicographic box mesh comes out unchanged and gets no inner
// context).  sem_pcg then gathers b and x0 into the inner order (4 KB blocks), runs the very same loop there -- where a
// node's copies are again close in memory, so the gather-scatter finds them in L2 and within TLB reach -- and scatters x
// back.  Everything else (sem_ax, sem_gs, sem_ax_gs, the accessors) stays on the caller-order context.
#include <stdlib.h>

#include <vector>

#include <cub/cub.cuh>

#include "sem_internal.h"

namespace {

__global__ void k_min_l2u(int64_t E, int p3, const int32_t* __restrict__ l2u, int32_t* __restrict__ key,
                          int32_t* __restrict__ val) {
    const int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (e >= E) return;
    int32_t m = l2u[e * p3];
    for (int t = 1; t < p3; ++t) { const int32_t v = l2u[e * p3 + t]; m = v < m ? v : m; }
    key[e] = m;                                   // rank of the smallest global id of the element
    val[e] = (int32_t)e;
}

// permuted inputs of the inner context, rebuilt from the canonical maps: gid = uniq_gid[l2u], flag = unique-node mask
__global__ void k_perm_inputs(int64_t E, int p3, const int32_t* __restrict__ perm, const int32_t* __restrict__ l2u,
                              const int64_t* __restrict__ uniq_gid, const uint8_t* __restrict__ mask_u,
                              const double* __restrict__ vert, int64_t* __restrict__ gid_p, uint8_t* __restrict__ dir_p,
                              double* __restrict__ vert_p) {
    for (int64_t q = blockIdx.x; q < E; q += gridDim.x) {
        const int64_t e = perm[q];
        for (int t = threadIdx.x; t < p3; t += blockDim.x) {
            const int32_t g = l2u[e * p3 + t];
            gid_p[q * p3 + t] = uniq_gid[g];
            if (dir_p) dir_p[q * p3 + t] = mask_u[g];
        }
        if (threadIdx.x < 24) vert_p[q * 24 + threadIdx.x] = vert[e * 24 + threadIdx.x];
    }
}

// dst[q][.] = src[perm[q]][.] (GATHER) or dst[perm[q]][.] = src[q][.] (scatter back), blocks of p3 doubles
template <bool GATHER>
__global__ void __launch_bounds__(256) k_perm_blocks(int64_t E, int p3, const int32_t* __restrict__ perm,
                                                     const double* __restrict__ src, double* __restrict__ dst) {
    for (int64_t q = blockIdx.x; q < E; q += gridDim.x) {
        const int64_t e = perm[q];
        for (int t = threadIdx.x; t < p3; t += blockDim.x) {
            if (GATHER) dst[q * p3 + t] = src[e * p3 + t];
            else dst[e * p3 + t] = src[q * p3 + t];
        }
    }
}

}  // namespace

void sem_inner_free(sem_ctx* c) {
    if (c->inner) { sem_ctx_destroy(c->inner); c->inner = nullptr; }
    cudaFree(c->d_perm); c->d_perm = nullptr;
    cudaFree(c->d_bi); c->d_bi = nullptr;
    cudaFree(c->d_xi); c->d_xi = nullptr;
    cudaGetLastError();
}

// Called at the end of sem_geom.  Decides whether the element order needs an inner context and builds it.
int sem_inner_build(sem_ctx* c, const double* node_xyz_host) {
    sem_inner_free(c);
    if (c->is_inner) return SEM_OK;
    const char* env = getenv("SEM_INNER");                       // "1": always, "0": never (tests, experiments)
    if (env && env[0] == '0') return SEM_OK;
    const bool force = env && env[0] == '1';
    if (!force && (double)c->nL * 8.0 < 256.0 * 1024 * 1024) return SEM_OK;      // the fields fit in (or near) L2 anyway
    cudaStream_t st = c->stream;
    const int64_t E = c->E;
    const int p3 = (int)c->p3;
    int32_t *d_key = nullptr, *d_val = nullptr, *d_key_s = nullptr;
    void* d_tmp = nullptr;
    auto drop = [&]() { cudaFree(d_key); cudaFree(d_val); cudaFree(d_key_s); cudaFree(d_tmp); };
    SEM_CUDA_OK(c, cudaMalloc((void**)&d_key, E * sizeof(int32_t)));
    SEM_CUDA_OK(c, cudaMalloc((void**)&d_val, E * sizeof(int32_t)));
    SEM_CUDA_OK(c, cudaMalloc((void**)&d_key_s, E * sizeof(int32_t)));
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_perm, E * sizeof(int32_t)));
    k_min_l2u<<<(unsigned)((E + 127) / 128), 128, 0, st>>>(E, p3, c->d_l2u, d_key, d_val);
    size_t tb = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, tb, d_key, d_key_s, d_val, c->d_perm, (int)E, 0, 32, st);
    SEM_CUDA_OK(c, cudaMalloc(&d_tmp, tb ? tb : 1));
    SEM_CUDA_OK(c, cub::DeviceRadixSort::SortPairs(d_tmp, tb, d_key, d_key_s, d_val, c->d_perm, (int)E, 0, 32, st));
    std::vector<int32_t> perm(E);
    SEM_CUDA_OK(c, cudaMemcpyAsync(perm.data(), c->d_perm, E * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    drop();
    // disorder: elements that sit further than E / 16 from their place in the sorted order
    int64_t far = 0;
    for (int64_t q = 0; q < E; ++q) far += llabs((long long)perm[q] - (long long)q) > E / 16;
    if (!force && far * 4 < E) { cudaFree(c->d_perm); c->d_perm = nullptr; return SEM_OK; }
    // ---- permuted inputs, then an ordinary context over them ----
    int64_t* d_gid_p = nullptr;
    uint8_t* d_dir_p = nullptr;
    double* d_vert_p = nullptr;
    SEM_CUDA_OK(c, cudaMalloc((void**)&d_gid_p, c->nL * sizeof(int64_t)));
    if (c->has_mask) SEM_CUDA_OK(c, cudaMalloc((void**)&d_dir_p, c->nL));
    SEM_CUDA_OK(c, cudaMalloc((void**)&d_vert_p, E * 24 * sizeof(double)));
    k_perm_inputs<<<(unsigned)(E < 65535 * 16 ? E : 65535 * 16), 128, 0, st>>>(E, p3, c->d_perm, c->d_l2u, c->d_uniq_gid, c->d_mask_u,
                                                                              c->d_vert, d_gid_p, d_dir_p, d_vert_p);
    std::vector<double> vert_p(E * 24);
    std::vector<uint8_t> dir_p(c->has_mask ? c->nL : 0);
    cudaError_t e1 = cudaMemcpyAsync(vert_p.data(), d_vert_p, E * 24 * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e1 == cudaSuccess && c->has_mask) e1 = cudaMemcpyAsync(dir_p.data(), d_dir_p, c->nL, cudaMemcpyDeviceToHost, st);
    if (e1 == cudaSuccess) e1 = cudaStreamSynchronize(st);
    cudaFree(d_vert_p);
    cudaFree(d_dir_p);
    if (e1 != cudaSuccess) { cudaFree(d_gid_p); return sem_fail(c, SEM_ECUDA, "inner context: %s", cudaGetErrorString(e1)); }
    sem_ctx* in = nullptr;
    int rc = sem_mesh_setup_impl(&in, E, c->N, vert_p.data(), d_gid_p, c->has_mask ? dir_p.data() : nullptr, (void*)st, true);
    cudaFree(d_gid_p);
    if (rc == SEM_OK) {
        std::vector<double> xyz_p;
        if (node_xyz_host) {                                         // isoparametric geometry: permute the coordinates too
            xyz_p.resize((size_t)c->nL * 3);
            for (int64_t q = 0; q < E; ++q)
                for (int64_t t = 0; t < (int64_t)p3 * 3; ++t) xyz_p[q * p3 * 3 + t] = node_xyz_host[(int64_t)perm[q] * p3 * 3 + t];
        }
        rc = sem_geom(in, node_xyz_host ? xyz_p.data() : nullptr, c->gmode, c->with_mass ? 1 : 0);
    }
    if (rc != SEM_OK) {
        sem_fail(c, rc, "inner context: %s", in ? in->err.c_str() : "allocation failed");
        if (in) sem_ctx_destroy(in);
        cudaFree(c->d_perm); c->d_perm = nullptr;
        return rc;
    }
    c->inner = in;
    return SEM_OK;
}

// sem_pcg through the inner context: gather b, x0; solve; scatter x; hand the history over
int sem_inner_pcg(sem_ctx* c, const double* b, double* x, double tol, int maxit, int* iters_out, double* relres_out) {
    sem_ctx* in = c->inner;
    cudaStream_t st = c->stream;
    if (!c->d_bi) SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_bi, c->nL * sizeof(double)));
    if (!c->d_xi) SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_xi, c->nL * sizeof(double)));
    const unsigned grid = (unsigned)(c->E < (int64_t)c->num_sms * 16 ? c->E : (int64_t)c->num_sms * 16);
    k_perm_blocks<true><<<grid, 256, 0, st>>>(c->E, (int)c->p3, c->d_perm, b, c->d_bi);
    k_perm_blocks<true><<<grid, 256, 0, st>>>(c->E, (int)c->p3, c->d_perm, x, c->d_xi);
    in->lambda = c->lambda;
    int rc = sem_pcg(in, c->d_bi, c->d_xi, tol, maxit, iters_out, relres_out);
    if (rc) return sem_fail(c, rc, "%s", in->err.c_str());
    k_perm_blocks<false><<<grid, 256, 0, st>>>(c->E, (int)c->p3, c->d_perm, c->d_xi, x);
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    delete[] c->h_hist;
    c->h_hist = new double[in->hist_n];
    c->hist_n = in->hist_n;
    for (int i = 0; i < in->hist_n; ++i) c->h_hist[i] = in->h_hist[i];
    return SEM_OK;
}
