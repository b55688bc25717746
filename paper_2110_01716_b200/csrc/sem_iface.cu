// sem_iface.cu — NEXT-4: the device side of the gather-scatter ACROSS ranks when the elements are
// partitioned over several GPUs.  P:119 "exchange-and-sum of shared interface values"; P:89 (overlap with interior work).
// A rank owns a contiguous block of elements and its own context; sem_gs sums the copies inside the rank; for the nodes
// that also live on other ranks (resolved once from the global ids, paper_2110_01716_b200/sharded.py) every rank
//   packs      buf[q] = w[first local copy of node uniq[q]]              (the rank-local sum, one value per shared node)
//   exchanges  the buffers with the ranks that share those nodes        (NCCL send/recv or peer copies: plumbing)
//   adds       w[every local copy of node uniq[q]] += buf_from_rank[q]
// in ascending rank order, so every rank ends with the same total on every copy.  Both kernels are gathers/scatters
// through the canonical maps (seg_off, seg_idx) of the context; no atomics (a node appears once per list).
#include "sem_internal.h"

namespace {

template <typename T>
__global__ void __launch_bounds__(256) k_iface_pack(int64_t n, const int32_t* __restrict__ uniq,
                                                    const int64_t* __restrict__ seg_off,
                                                    const int32_t* __restrict__ seg_idx, const T* __restrict__ w,
                                                    T* __restrict__ buf) {
    for (int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; q < n; q += (int64_t)gridDim.x * blockDim.x)
        buf[q] = w[seg_idx[seg_off[uniq[q]]]];
}

template <typename T>
__global__ void __launch_bounds__(256) k_iface_add(int64_t n, const int32_t* __restrict__ uniq,
                                                   const int64_t* __restrict__ seg_off,
                                                   const int32_t* __restrict__ seg_idx, const uint8_t* __restrict__ mask_u,
                                                   const T* __restrict__ buf, T* __restrict__ w) {
    for (int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; q < n; q += (int64_t)gridDim.x * blockDim.x) {
        const int32_t g = uniq[q];
        if (mask_u && mask_u[g]) continue;                  // Dirichlet node: stays zero on every rank
        const T v = buf[q];
        for (int64_t s = seg_off[g]; s < seg_off[g + 1]; ++s) w[seg_idx[s]] += v;
    }
}

int check(sem_ctx* c, const void* uniq, int64_t n, const void* w, const void* buf, sem_prec prec, const char* who) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (n < 0 || (n > 0 && (!uniq || !w || !buf))) return sem_fail(c, SEM_EINVAL, "%s: NULL pointer or n < 0", who);
    if (prec != SEM_F64 && prec != SEM_F32) return sem_fail(c, SEM_EINVAL, "%s: bad sem_prec", who);
    if (!c->d_seg_off) return sem_fail(c, SEM_ESTATE, "%s on a context whose setup failed", who);
    return SEM_OK;
}

}  // namespace

extern "C" int sem_iface_pack(sem_ctx* c, const int32_t* uniq, int64_t n, const void* w, void* buf, sem_prec prec) {
    int rc = check(c, uniq, n, w, buf, prec, "sem_iface_pack");
    if (rc || n == 0) return rc;
    const unsigned grid = (unsigned)((n + 255) / 256 < (int64_t)c->num_sms * 8 ? (n + 255) / 256 : (int64_t)c->num_sms * 8);
    if (prec == SEM_F64)
        k_iface_pack<double><<<grid, 256, 0, c->stream>>>(n, uniq, c->d_seg_off, c->d_seg_idx, (const double*)w, (double*)buf);
    else
        k_iface_pack<float><<<grid, 256, 0, c->stream>>>(n, uniq, c->d_seg_off, c->d_seg_idx, (const float*)w, (float*)buf);
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

extern "C" int sem_iface_add(sem_ctx* c, const int32_t* uniq, int64_t n, const void* buf, void* w, sem_prec prec) {
    int rc = check(c, uniq, n, w, buf, prec, "sem_iface_add");
    if (rc || n == 0) return rc;
    const unsigned grid = (unsigned)((n + 255) / 256 < (int64_t)c->num_sms * 8 ? (n + 255) / 256 : (int64_t)c->num_sms * 8);
    const uint8_t* mk = c->has_mask ? c->d_mask_u : nullptr;
    if (prec == SEM_F64)
        k_iface_add<double><<<grid, 256, 0, c->stream>>>(n, uniq, c->d_seg_off, c->d_seg_idx, mk, (const double*)buf, (double*)w);
    else
        k_iface_add<float><<<grid, 256, 0, c->stream>>>(n, uniq, c->d_seg_off, c->d_seg_idx, mk, (const float*)buf, (float*)w);
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}
