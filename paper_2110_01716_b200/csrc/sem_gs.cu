// sem_gs.cu — a6 + a7: gather-scatter QQ^T (op = add) in place on a local-layout field, plus the Dirichlet mask.
// P:119 "exchange-and-sum of shared interface values"; O5: every copy of a unique node receives the sum over its
// copies, accumulated in ascending local index (the same order as the CPU oracle, so FP results are bit-identical).
// Only nodes with multiplicity > 1 are touched (compressed map sh_off/sh_idx built in sem_maps.cu); no atomics.
#include "sem_internal.h"

namespace {

template <typename T>
__global__ void __launch_bounds__(256) k_gs(int32_t Us, const int32_t* __restrict__ sh_off,
                                            const int32_t* __restrict__ sh_idx,
                                            const uint8_t* __restrict__ sh_masked, T* __restrict__ w,
                                            int32_t n_mask1, const int32_t* __restrict__ mask1_idx) {
    const int32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < Us) {
        const int32_t b = sh_off[t], e = sh_off[t + 1];
        T s;
        if (e - b == 2) {                      // a face node: the common case, both loads in flight together
            const int32_t l0 = sh_idx[b], l1 = sh_idx[b + 1];
            const T a0 = w[l0], a1 = w[l1];
            s = a0 + a1;
            if (sh_masked && sh_masked[t]) s = T(0);
            w[l0] = s; w[l1] = s;
        } else if (e - b == 4) {               // an edge node
            const int32_t l0 = sh_idx[b], l1 = sh_idx[b + 1], l2 = sh_idx[b + 2], l3 = sh_idx[b + 3];
            const T a0 = w[l0], a1 = w[l1], a2 = w[l2], a3 = w[l3];
            s = ((a0 + a1) + a2) + a3;
            if (sh_masked && sh_masked[t]) s = T(0);
            w[l0] = s; w[l1] = s; w[l2] = s; w[l3] = s;
        } else {
            s = T(0);
            for (int32_t q = b; q < e; ++q) s += w[sh_idx[q]];
            if (sh_masked && sh_masked[t]) s = T(0);
            for (int32_t q = b; q < e; ++q) w[sh_idx[q]] = s;
        }
    } else if (t - Us < n_mask1) {
        w[mask1_idx[t - Us]] = T(0);           // masked nodes that are not shared
    }
}

}  // namespace

int sem_launch_gs(sem_ctx* c, void* w, sem_prec prec, bool apply_mask) {
    const bool m = apply_mask && c->has_mask;
    const int64_t total = c->Us + (m ? c->n_mask1 : 0);
    if (total == 0) return SEM_OK;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    if (prec == SEM_F64)
        k_gs<double><<<blocks, 256, 0, c->stream>>>((int32_t)c->Us, c->d_sh_off, c->d_sh_idx, m ? c->d_sh_masked : nullptr,
                                                    (double*)w, m ? (int32_t)c->n_mask1 : 0, c->d_mask1_idx);
    else
        k_gs<float><<<blocks, 256, 0, c->stream>>>((int32_t)c->Us, c->d_sh_off, c->d_sh_idx, m ? c->d_sh_masked : nullptr,
                                                   (float*)w, m ? (int32_t)c->n_mask1 : 0, c->d_mask1_idx);
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}
