// sem_gs.cu — a6 + a7: gather-scatter QQ^T (op = add) in place on a local-layout field, plus the Dirichlet mask.
// P:119 "exchange-and-sum of shared interface values"; O5: every copy of a unique node receives the sum over its
// copies, accumulated in ascending local index (the same order as the CPU oracle, so FP results are bit-identical).
// Only nodes with multiplicity > 1 are touched; no atomics on data.
//
// The work is not bandwidth-bound (at config 2 the field sits in L2 after the Ax kernel): it is bound by dependent
// memory round trips and by L1 sector look-ups of scattered 8-byte accesses.  So the segments are pre-resolved at
// setup (sem_maps.cu, sem_build_owner_lists) into fixed-format records, sorted by OWNER element group (the group that
// holds the node's last copy),
//   pair (l0 | maskbit, l1)             2 copies     (l1 = -1: an unshared Dirichlet node, only zeroed)
//   quad (l0 | maskbit, l1, l2, l3|-1)  3-4 copies
//   big  (offset into sh_idx, count | maskbit)       > 4 copies
// and a thread handles PPT pairs (or one quad / big) at a time: one coalesced record load, then all value loads
// together, then the stores: two dependent round trips instead of three (offsets -> indices -> values).
#include "sem_gs_dev.cuh"
#include "sem_internal.h"

namespace {

using namespace semgs;

// ---------------------------------------------------------------------------------------------------------------
// Stand-alone kernel (sem_gs, and sem_ax_gs where the single-pass path does not apply).  The grid is ONE wave
// (<= resident CTAs of the device) and every CTA owns the same share of every record class: no tail, no imbalance.
// ---------------------------------------------------------------------------------------------------------------
constexpr int NT = 256, GS_CTAS = 5;      // threads per CTA, resident CTAs per SM (48 registers, no spills)

template <typename T, bool MASK>
__global__ void __launch_bounds__(NT, GS_CTAS) k_gs_records(int32_t n_pair, const int2* __restrict__ pair, int32_t n_quad,
                                                   const int4* __restrict__ quad, int32_t n_big,
                                                   const int2* __restrict__ big, const int32_t* __restrict__ sh_idx,
                                                   T* __restrict__ w) {
    // every CTA takes the same share of every record class (contiguous, whole 32-record rows): balanced by construction
    const int32_t b = blockIdx.x, nb = gridDim.x;
    const int32_t pp = ((n_pair + nb - 1) / nb + 31) & ~31, pq = ((n_quad + nb - 1) / nb + 31) & ~31,
                  pg = (n_big + nb - 1) / nb;
    const int64_t bp = (int64_t)b * pp, bq = (int64_t)b * pq, bg = (int64_t)b * pg;
    if (bp < n_pair) gs_pairs<T, MASK, false, NT>(pair, (int32_t)bp + threadIdx.x, min(n_pair, (int32_t)bp + pp), w);
    if (bq < n_quad) gs_quads<T, MASK, false, NT>(quad, (int32_t)bq + threadIdx.x, min(n_quad, (int32_t)bq + pq), w);
    if (bg < n_big) gs_bigs<T, MASK, false, NT>(big, sh_idx, (int32_t)bg + threadIdx.x, min(n_big, (int32_t)bg + pg), w);
}

}  // namespace

int sem_launch_gs(sem_ctx* c, void* w, sem_prec prec, bool apply_mask) {
    const bool m = apply_mask && c->has_mask;
    const int32_t np = (int32_t)c->n_pair, nq = (int32_t)c->n_quad, nb = (int32_t)c->n_big;
    if (np + nq + nb == 0) return SEM_OK;
    // one wave of CTAs (8 x 256 threads per SM), fewer when there is less than one row of PPT pairs per thread
    const double ops = 4.0 * np + 8.0 * nq + 16.0 * nb;
    int64_t blocks = (int64_t)(ops / (4.0 * NT * PPT)) + 1;
    const int64_t cap = (int64_t)c->num_sms * GS_CTAS;
    if (blocks > cap) blocks = cap;
    blocks = (blocks + c->num_sms - 1) / c->num_sms * c->num_sms;      // same number of CTAs on every SM
#define SEM_GS_LAUNCH(T, M)                                                                                      \
    k_gs_records<T, M><<<(unsigned)blocks, NT, 0, c->stream>>>(np, c->d_own_pair, nq, c->d_own_quad, nb,          \
                                                                c->d_own_big, c->d_sh_idx, (T*)w)
    if (prec == SEM_F64) { if (m) SEM_GS_LAUNCH(double, true); else SEM_GS_LAUNCH(double, false); }
    else { if (m) SEM_GS_LAUNCH(float, true); else SEM_GS_LAUNCH(float, false); }
#undef SEM_GS_LAUNCH
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}
