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
#include "sem_internal.h"

namespace {

constexpr int32_t IDX = 0x7fffffff;
constexpr int PPT = 4;           // pairs per thread in flight

// COHERENT: read values with ld.relaxed.gpu (from L2): they were written by another, still running, kernel
template <typename T, bool COHERENT>
__device__ __forceinline__ T ld_val(const T* p) {
    if constexpr (!COHERENT) return *p;
    else if constexpr (sizeof(T) == 8) {
        double v;
        asm volatile("ld.relaxed.gpu.global.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
        return v;
    } else {
        float v;
        asm volatile("ld.relaxed.gpu.global.f32 %0, [%1];" : "=f"(v) : "l"(p) : "memory");
        return v;
    }
}

// records [first, end) with stride NTH between the records of one thread
template <typename T, bool MASK, bool COHERENT, int NTH, int PP = PPT>
__device__ __forceinline__ void gs_pairs(const int2* __restrict__ pair, int32_t first, int32_t end, T* __restrict__ w) {
    for (int32_t base = first; base < end; base += NTH * PP) {
        int2 r[PP];
#pragma unroll
        for (int q = 0; q < PP; ++q) {
            const int32_t t = base + q * NTH;
            r[q] = t < end ? pair[t] : make_int2(0, -2);        // -2: nothing to do
        }
        T v0[PP], v1[PP];
#pragma unroll
        for (int q = 0; q < PP; ++q) {
            v0[q] = r[q].y >= 0 ? ld_val<T, COHERENT>(w + (r[q].x & IDX)) : T(0);
            v1[q] = r[q].y >= 0 ? ld_val<T, COHERENT>(w + r[q].y) : T(0);
        }
#pragma unroll
        for (int q = 0; q < PP; ++q) {
            if (r[q].y >= 0) {
                T s = v0[q] + v1[q];
                if (MASK && r[q].x < 0) s = T(0);
                w[r[q].x & IDX] = s;
                w[r[q].y] = s;
            } else if (MASK && r[q].y == -1) {
                w[r[q].x & IDX] = T(0);
            }
        }
    }
}

template <typename T, bool MASK, bool COHERENT, int NTH>
__device__ __forceinline__ void gs_quads(const int4* __restrict__ quad, int32_t first, int32_t end, T* __restrict__ w) {
    for (int32_t t = first; t < end; t += NTH) {
        const int4 r = quad[t];
        const int32_t l0 = r.x & IDX;
        const T a0 = ld_val<T, COHERENT>(w + l0), a1 = ld_val<T, COHERENT>(w + r.y), a2 = ld_val<T, COHERENT>(w + r.z);
        const T a3 = r.w >= 0 ? ld_val<T, COHERENT>(w + r.w) : T(0);
        T s = (a0 + a1) + a2;
        if (r.w >= 0) s += a3;
        if (MASK && r.x < 0) s = T(0);
        w[l0] = s; w[r.y] = s; w[r.z] = s;
        if (r.w >= 0) w[r.w] = s;
    }
}

template <typename T, bool MASK, bool COHERENT, int NTH>
__device__ __forceinline__ void gs_bigs(const int2* __restrict__ big, const int32_t* __restrict__ sh_idx, int32_t first,
                                        int32_t end, T* __restrict__ w) {
    for (int32_t t = first; t < end; t += NTH) {
        const int2 r = big[t];
        const int32_t cnt = r.y & IDX;
        // the first 8 copies (a corner of a hexahedral mesh has 8) with all loads in flight together
        int32_t id[8];
        T v[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) id[q] = q < cnt ? __ldg(&sh_idx[r.x + q]) : -1;
#pragma unroll
        for (int q = 0; q < 8; ++q) v[q] = id[q] >= 0 ? ld_val<T, COHERENT>(w + id[q]) : T(0);
        T s = v[0];
#pragma unroll
        for (int q = 1; q < 8; ++q) if (id[q] >= 0) s += v[q];
        for (int32_t q = 8; q < cnt; ++q) s += ld_val<T, COHERENT>(w + sh_idx[r.x + q]);
        if (MASK && r.y < 0) s = T(0);
#pragma unroll
        for (int q = 0; q < 8; ++q) if (id[q] >= 0) w[id[q]] = s;
        for (int32_t q = 8; q < cnt; ++q) w[sh_idx[r.x + q]] = s;
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Stand-alone kernel (sem_gs, and sem_ax_gs where the single-pass path does not apply).  The grid is ONE wave
// (<= resident CTAs of the device) and every CTA owns the same share of every record class: no tail, no imbalance.
// ---------------------------------------------------------------------------------------------------------------
constexpr int NT = 256;

template <typename T, bool MASK>
__global__ void __launch_bounds__(NT) k_gs_records(int32_t n_pair, const int2* __restrict__ pair, int32_t n_quad,
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

// ---------------------------------------------------------------------------------------------------------------
// Single-pass Ax+gs: gather-scatter WORKERS that run concurrently with the operator kernel (sem_ax.cu, FUSE = true).
// The worker grid is a programmatic dependent launch: it starts as soon as every CTA of the operator grid is running
// (those CTAs execute griddepcontrol.launch_dependents first thing), on the SM resources the operator grid leaves
// free: the operator is launched with one CTA per SM fewer than fit, which frees 4096 registers on each of two SM
// sub-partitions -- room for exactly one 2-warp worker CTA of <= 128 registers per thread.  The operator is
// HBM-bound and the gather-scatter is bound by L1 sector look-ups and L2 round trips, so the two overlap.
//   * operator CTA b applies element groups b, b + n_ax, ... ("waves" of n_ax groups) and publishes
//     red.release.gpu.add(done[v]) after the stores of its group of wave v (sem_ax.cu);
//   * worker CTA c owns chunks c, c + #workers, ... of GCH consecutive OWNER groups (a shared node is owned by the
//     group holding its last copy, so every other copy lives in a lower group).  For each chunk it waits (acquire)
//     until the wave of the chunk's last group is complete -- by the ascending round-robin order every lower group is
//     then complete too -- sums the chunk's records in ascending local index (O5) and writes every copy;
//   * the records of the NEXT chunk are prefetched into shared memory (cp.async) while the values of the current one
//     are in flight, so a chunk costs about two dependent L2 round trips.
// The operator never waits on a worker, and every operator CTA is resident before the first worker starts: no
// deadlock.  A node is written by its own group before that group's done-increment and by exactly one worker thread
// after it.  The last worker CTA to leave zeroes the counters for the next launch.
// ---------------------------------------------------------------------------------------------------------------
constexpr int WNT = 64;          // worker threads per CTA
constexpr int GCH = 4;           // owner groups per chunk
constexpr int WPPT = 8;          // pairs per worker thread in flight
constexpr int PCAP = 1024, QCAP = 192, BCAP = 32;     // records per class staged in shared memory (rest: global)

__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void cp_async_8(void* dst_smem, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src)
                 : "memory");
}
__device__ __forceinline__ void cp_async_16(void* dst_smem, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src)
                 : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

struct WorkerSmem {
    int4 sq[2][QCAP];
    int2 sp[2][PCAP];
    int2 sb[2][BCAP];
};

template <typename T, bool MASK>
__global__ void __launch_bounds__(WNT, 8) k_gs_worker(int32_t ngroups, int32_t n_ax, const int4* __restrict__ goff,
                                                      const int2* __restrict__ pair, const int4* __restrict__ quad,
                                                      const int2* __restrict__ big, const int32_t* __restrict__ sh_idx,
                                                      uint32_t* __restrict__ ctr, const int* __restrict__ skip_flag,
                                                      T* __restrict__ w) {
    if (skip_flag && *skip_flag) return;
    __shared__ WorkerSmem sm;
    const int tid = threadIdx.x;
    const int32_t nchunks = (ngroups + GCH - 1) / GCH;
    const int32_t stride = (int32_t)gridDim.x;
    auto prefetch = [&](int buf, const int4& a, const int4& b) {
        const int32_t np = min(b.y - a.y, PCAP), nq = min(b.z - a.z, QCAP), nb = min(b.w - a.w, BCAP);
        for (int32_t t = tid; t < np; t += WNT) cp_async_8(&sm.sp[buf][t], pair + a.y + t);
        for (int32_t t = tid; t < nq; t += WNT) cp_async_16(&sm.sq[buf][t], quad + a.z + t);
        for (int32_t t = tid; t < nb; t += WNT) cp_async_8(&sm.sb[buf][t], big + a.w + t);
    };
    int32_t q = (int32_t)blockIdx.x;
    int cur = 0;
    int4 o0 = make_int4(0, 0, 0, 0), o1 = o0;
    if (q < nchunks) {
        o0 = __ldg(goff + q * GCH);
        o1 = __ldg(goff + min(ngroups, (q + 1) * GCH));
        prefetch(0, o0, o1);
    }
    while (q < nchunks) {
        const int32_t qn = q + stride;
        int4 n0 = o0, n1 = o0;
        if (qn < nchunks) {                       // offsets of the next chunk: in flight during the poll
            n0 = __ldg(goff + qn * GCH);
            n1 = __ldg(goff + min(ngroups, (qn + 1) * GCH));
        }
        const int32_t wave = (min(ngroups, (q + 1) * GCH) - 1) / n_ax;
        const uint32_t target = (uint32_t)min(n_ax, ngroups - wave * n_ax);
        if (tid == 0) while (ld_acquire_u32(ctr + SEM_CTR_DONE + SEM_CTR_STRIDE * wave) < target) __nanosleep(200);
        cp_async_wait_all();
        __syncthreads();                          // records of this chunk staged; its wave is complete
        if (qn < nchunks) prefetch(cur ^ 1, n0, n1);
        const int32_t np = o1.y - o0.y, nq = o1.z - o0.z, nb = o1.w - o0.w;
        gs_pairs<T, MASK, true, WNT, WPPT>(sm.sp[cur], tid, min(np, PCAP), w);
        gs_quads<T, MASK, true, WNT>(sm.sq[cur], tid, min(nq, QCAP), w);
        gs_bigs<T, MASK, true, WNT>(sm.sb[cur], sh_idx, tid, min(nb, BCAP), w);
        if (np > PCAP) gs_pairs<T, MASK, true, WNT, WPPT>(pair + o0.y, PCAP + tid, np, w);      // overflow: from global
        if (nq > QCAP) gs_quads<T, MASK, true, WNT>(quad + o0.z, QCAP + tid, nq, w);
        if (nb > BCAP) gs_bigs<T, MASK, true, WNT>(big + o0.w, sh_idx, BCAP + tid, nb, w);
        q = qn; o0 = n0; o1 = n1; cur ^= 1;
    }
    cp_async_wait_all();
    if (tid == 0) {
        const uint32_t ticket = atomicAdd(ctr + SEM_CTR_TICKET, 1u);
        if (ticket == gridDim.x - 1) {        // every other worker is done: nobody reads the counters any more
            const int32_t nwaves = (ngroups + n_ax - 1) / n_ax;
            for (int32_t v = 0; v < nwaves; ++v) ctr[SEM_CTR_DONE + SEM_CTR_STRIDE * v] = 0u;
            __threadfence();
            ctr[SEM_CTR_TICKET] = 0u;
        }
    }
}

}  // namespace

int sem_launch_gs(sem_ctx* c, void* w, sem_prec prec, bool apply_mask) {
    const bool m = apply_mask && c->has_mask;
    const int32_t np = (int32_t)c->n_pair, nq = (int32_t)c->n_quad, nb = (int32_t)c->n_big;
    if (np + nq + nb == 0) return SEM_OK;
    // one wave of CTAs (8 x 256 threads per SM), fewer when there is less than one row of PPT pairs per thread
    const double ops = 4.0 * np + 8.0 * nq + 16.0 * nb;
    int64_t blocks = (int64_t)(ops / (4.0 * NT * PPT)) + 1;
    const int64_t cap = (int64_t)c->num_sms * 8;
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

int sem_launch_gs_worker(sem_ctx* c, void* w, sem_prec prec, int32_t n_ax, int32_t ngroups, int32_t group_nodes,
                         const int* skip_flag) {
    (void)group_nodes;
    const bool m = c->has_mask;
    const int32_t nchunks = (ngroups + GCH - 1) / GCH;
    int64_t grid = c->num_sms;                  // one worker CTA fits beside the operator CTAs of an SM
    if (grid > nchunks) grid = nchunks;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(WNT);
    cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
#define SEM_GSW_LAUNCH(T, M)                                                                                       \
    SEM_CUDA_OK(c, cudaLaunchKernelEx(&cfg, k_gs_worker<T, M>, ngroups, n_ax, (const int4*)c->d_own_goff,          \
                                      (const int2*)c->d_own_pair, (const int4*)c->d_own_quad,                      \
                                      (const int2*)c->d_own_big, (const int32_t*)c->d_sh_idx, c->d_gs_flag,        \
                                      skip_flag, (T*)w))
    if (prec == SEM_F64) { if (m) SEM_GSW_LAUNCH(double, true); else SEM_GSW_LAUNCH(double, false); }
    else { if (m) SEM_GSW_LAUNCH(float, true); else SEM_GSW_LAUNCH(float, false); }
#undef SEM_GSW_LAUNCH
    return SEM_OK;
}
