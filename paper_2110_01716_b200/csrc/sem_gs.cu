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
                                                   T* __restrict__ w, const int* __restrict__ skip_flag) {
    if (skip_flag && *skip_flag) return;                 // the PCG loop has converged: every later launch is a no-op
    // every CTA takes the same share of every record class (contiguous, whole 32-record rows): balanced by construction
    const int32_t b = blockIdx.x, nb = gridDim.x;
    const int32_t pp = ((n_pair + nb - 1) / nb + 31) & ~31, pq = ((n_quad + nb - 1) / nb + 31) & ~31,
                  pg = (n_big + nb - 1) / nb;
    const int64_t bp = (int64_t)b * pp, bq = (int64_t)b * pq, bg = (int64_t)b * pg;
    if (bp < n_pair) gs_pairs<T, MASK, NT>(pair, (int32_t)bp + threadIdx.x, min(n_pair, (int32_t)bp + pp), w);
    if (bq < n_quad) gs_quads<T, MASK, NT>(quad, (int32_t)bq + threadIdx.x, min(n_quad, (int32_t)bq + pq), w);
    if (bg < n_big) gs_bigs<T, MASK, NT>(big, sh_idx, (int32_t)bg + threadIdx.x, min(n_big, (int32_t)bg + pg), w);
}

// ---------------------------------------------------------------------------------------------------------------
// Several fields in one launch (sem_gs_many; the paper's `gatherScatterMany`, Table 3: the three velocity
// components of the Helmholtz solves): a record is read once and applied to NF fields w + f * stride, with the
// value loads of all NF fields in flight together.  Same ascending-index sums per field, so each field is bit-identical
// to sem_gs applied to it alone.
// ---------------------------------------------------------------------------------------------------------------
template <typename T, bool MASK, int NF, bool INTER>
__global__ void __launch_bounds__(NT, 4) k_gs_records_many(int32_t n_pair, const int2* __restrict__ pair, int32_t n_quad,
                                                           const int4* __restrict__ quad, int32_t n_big,
                                                           const int2* __restrict__ big,
                                                           const int32_t* __restrict__ sh_idx, T* __restrict__ w,
                                                           int64_t stride, const int* __restrict__ skip_flag) {
    if (skip_flag && *skip_flag) return;
    // value of field f at local node l: planar fields w + f * stride, or node-interleaved [nL][NF]
    auto at = [&](int f, int32_t l) -> T& { return INTER ? w[(int64_t)l * NF + f] : w[f * stride + l]; };
    // all NF values of a node: interleaved fields whose NF values fill whole 16-byte words move as vectors
    constexpr bool VEC = INTER && (NF * sizeof(T)) % 16 == 0;
    constexpr int NV = VEC ? (int)(NF * sizeof(T) / 16) : 1;
    auto ldn = [&](int32_t l, T (&v)[NF]) {
        if constexpr (VEC) {
            const int4* src = reinterpret_cast<const int4*>(w + (int64_t)l * NF);
#pragma unroll
            for (int q = 0; q < NV; ++q) reinterpret_cast<int4*>(v)[q] = src[q];
        } else {
#pragma unroll
            for (int f = 0; f < NF; ++f) v[f] = at(f, l);
        }
    };
    auto stn = [&](int32_t l, const T (&v)[NF]) {
        if constexpr (VEC) {
            int4* dst = reinterpret_cast<int4*>(w + (int64_t)l * NF);
#pragma unroll
            for (int q = 0; q < NV; ++q) dst[q] = reinterpret_cast<const int4*>(v)[q];
        } else {
#pragma unroll
            for (int f = 0; f < NF; ++f) at(f, l) = v[f];
        }
    };
    const int32_t b = blockIdx.x, nb = gridDim.x;
    const int32_t pp = ((n_pair + nb - 1) / nb + 31) & ~31, pq = ((n_quad + nb - 1) / nb + 31) & ~31,
                  pg = (n_big + nb - 1) / nb;
    const int64_t bp = (int64_t)b * pp, bq = (int64_t)b * pq, bg = (int64_t)b * pg;
    constexpr int PP = 2;                                     // pairs per thread and pass: PP x NF x 2 loads in flight
    if (bp < n_pair) {
        const int32_t end = min(n_pair, (int32_t)bp + pp);
        for (int32_t base = (int32_t)bp + threadIdx.x; base < end; base += NT * PP) {
            int2 r[PP];
#pragma unroll
            for (int q = 0; q < PP; ++q) {
                const int32_t t = base + q * NT;
                r[q] = t < end ? pair[t] : make_int2(0, -2);
            }
            alignas(16) T v0[PP][NF], v1[PP][NF];
#pragma unroll
            for (int q = 0; q < PP; ++q) {
                if (r[q].y >= 0) { ldn(r[q].x & IDX, v0[q]); ldn(r[q].y, v1[q]); }
            }
#pragma unroll
            for (int q = 0; q < PP; ++q) {
                if (r[q].y >= 0) {
#pragma unroll
                    for (int f = 0; f < NF; ++f) {
                        T s = v0[q][f] + v1[q][f];
                        if (MASK && r[q].x < 0) s = T(0);
                        v0[q][f] = s;
                    }
                    stn(r[q].x & IDX, v0[q]);
                    stn(r[q].y, v0[q]);
                } else if (MASK && r[q].y == -1) {
#pragma unroll
                    for (int f = 0; f < NF; ++f) v0[q][f] = T(0);
                    stn(r[q].x & IDX, v0[q]);
                }
            }
        }
    }
    if (bq < n_quad) {
        const int32_t end = min(n_quad, (int32_t)bq + pq);
        for (int32_t t = (int32_t)bq + threadIdx.x; t < end; t += NT) {
            const int4 r = quad[t];
            const int32_t l0 = r.x & IDX;
            alignas(16) T a[4][NF];
            ldn(l0, a[0]); ldn(r.y, a[1]); ldn(r.z, a[2]);
            if (r.w >= 0) ldn(r.w, a[3]);
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                T s = (a[0][f] + a[1][f]) + a[2][f];
                if (r.w >= 0) s += a[3][f];
                if (MASK && r.x < 0) s = T(0);
                a[0][f] = s;
            }
            stn(l0, a[0]); stn(r.y, a[0]); stn(r.z, a[0]);
            if (r.w >= 0) stn(r.w, a[0]);
        }
    }
    if (bg < n_big)                                           // rare (> 4 copies): field by field
        for (int f = 0; f < NF; ++f) {
            if (INTER) gs_bigs<T, MASK, NT, NF>(big, sh_idx, (int32_t)bg + threadIdx.x, min(n_big, (int32_t)bg + pg), w + f);
            else gs_bigs<T, MASK, NT>(big, sh_idx, (int32_t)bg + threadIdx.x, min(n_big, (int32_t)bg + pg), w + f * stride);
        }
}

}  // namespace

static int launch_records(sem_ctx* c, void* w, sem_prec prec, bool m, const int* skip_flag, int32_t p0, int32_t np,
                          int32_t q0, int32_t nq, int32_t b0, int32_t nb) {
    if (np + nq + nb == 0) return SEM_OK;
    // one wave of CTAs (8 x 256 threads per SM), fewer when there is less than one row of PPT pairs per thread
    const double ops = 4.0 * np + 8.0 * nq + 16.0 * nb;
    int64_t blocks = (int64_t)(ops / (4.0 * NT * PPT)) + 1;
    const int64_t cap = (int64_t)c->num_sms * GS_CTAS;
    if (blocks > cap) blocks = cap;
    blocks = (blocks + c->num_sms - 1) / c->num_sms * c->num_sms;      // same number of CTAs on every SM
#define SEM_GS_LAUNCH(T, M)                                                                                      \
    k_gs_records<T, M><<<(unsigned)blocks, NT, 0, c->stream>>>(np, c->d_own_pair + p0, nq, c->d_own_quad + q0, nb, \
                                                                c->d_own_big + b0, c->d_sh_idx, (T*)w, skip_flag)
    if (prec == SEM_F64) { if (m) SEM_GS_LAUNCH(double, true); else SEM_GS_LAUNCH(double, false); }
    else { if (m) SEM_GS_LAUNCH(float, true); else SEM_GS_LAUNCH(float, false); }
#undef SEM_GS_LAUNCH
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

int sem_launch_gs(sem_ctx* c, void* w, sem_prec prec, bool apply_mask, const int* skip_flag) {
    return launch_records(c, w, prec, apply_mask && c->has_mask, skip_flag, 0, (int32_t)c->n_pair, 0, (int32_t)c->n_quad, 0,
                          (int32_t)c->n_big);
}

// the records owned by the element groups of chunk `chunk` (sem_ctx::chunk_e0 / chunk_rec)
int sem_launch_gs_range(sem_ctx* c, void* w, sem_prec prec, bool apply_mask, const int* skip_flag, int chunk) {
    const int32_t *P = c->chunk_rec[0].data(), *Q = c->chunk_rec[1].data(), *B = c->chunk_rec[2].data();
    return launch_records(c, w, prec, apply_mask && c->has_mask, skip_flag, P[chunk], P[chunk + 1] - P[chunk], Q[chunk],
                          Q[chunk + 1] - Q[chunk], B[chunk], B[chunk + 1] - B[chunk]);
}

// nf = 2, 3 or 4 fields at w + f * stride (values of T) in one launch
int sem_launch_gs_many(sem_ctx* c, void* w, int nf, int64_t stride, sem_prec prec, bool apply_mask,
                       const int* skip_flag) {
    const bool m = apply_mask && c->has_mask;
    const int32_t np = (int32_t)c->n_pair, nq = (int32_t)c->n_quad, nb = (int32_t)c->n_big;
    if (np + nq + nb == 0) return SEM_OK;
    const double ops = (4.0 * np + 8.0 * nq + 16.0 * nb) * nf;
    int64_t blocks = (int64_t)(ops / (4.0 * NT * PPT)) + 1;
    const int64_t cap = (int64_t)c->num_sms * 4;
    if (blocks > cap) blocks = cap;
    blocks = (blocks + c->num_sms - 1) / c->num_sms * c->num_sms;
    const bool inter = stride == 1;                              // node-interleaved fields [nL][nf]
#define SEM_GSM_LAUNCH(T, M, NF, I)                                                                               \
    k_gs_records_many<T, M, NF, I><<<(unsigned)blocks, NT, 0, c->stream>>>(np, c->d_own_pair, nq, c->d_own_quad, nb, \
                                                                            c->d_own_big, c->d_sh_idx, (T*)w, stride, skip_flag)
#define SEM_GSM_I(T, M, NF)                                                                                       \
    do { if (inter) SEM_GSM_LAUNCH(T, M, NF, true); else SEM_GSM_LAUNCH(T, M, NF, false); } while (0)
#define SEM_GSM_NF(T, M)                                                                                          \
    do {                                                                                                          \
        if (nf == 2) SEM_GSM_I(T, M, 2);                                                                          \
        else if (nf == 3) SEM_GSM_I(T, M, 3);                                                                     \
        else SEM_GSM_I(T, M, 4);                                                                                  \
    } while (0)
    if (prec == SEM_F64) { if (m) SEM_GSM_NF(double, true); else SEM_GSM_NF(double, false); }
    else { if (m) SEM_GSM_NF(float, true); else SEM_GSM_NF(float, false); }
#undef SEM_GSM_NF
#undef SEM_GSM_I
#undef SEM_GSM_LAUNCH
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}
