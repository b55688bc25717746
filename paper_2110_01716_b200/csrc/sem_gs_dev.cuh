// sem_gs_dev.cuh — device-side record processing of the gather-scatter (a6 + a7) used by the kernels of sem_gs.cu.
// See sem_gs.cu for the record formats; sums run in ascending local index (O5), so results are bit-identical to the
// oracle's.
#pragma once
#include <stdint.h>

namespace semgs {

constexpr int32_t IDX = 0x7fffffff;
constexpr int PPT = 4;           // pairs per thread in flight

// records [first, end) with stride NTH between the records of one thread
template <typename T, bool MASK, int NTH, int PP = PPT>
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
            v0[q] = r[q].y >= 0 ? w[(r[q].x & IDX)] : T(0);
            v1[q] = r[q].y >= 0 ? w[r[q].y] : T(0);
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

template <typename T, bool MASK, int NTH>
__device__ __forceinline__ void gs_quads(const int4* __restrict__ quad, int32_t first, int32_t end, T* __restrict__ w) {
    for (int32_t t = first; t < end; t += NTH) {
        const int4 r = quad[t];
        const int32_t l0 = r.x & IDX;
        const T a0 = w[l0], a1 = w[r.y], a2 = w[r.z];
        const T a3 = r.w >= 0 ? w[r.w] : T(0);
        T s = (a0 + a1) + a2;
        if (r.w >= 0) s += a3;
        if (MASK && r.x < 0) s = T(0);
        w[l0] = s; w[r.y] = s; w[r.z] = s;
        if (r.w >= 0) w[r.w] = s;
    }
}

// NSTR: distance between consecutive nodes in values of T (1; NF for node-interleaved fields, w pointing at field f)
template <typename T, bool MASK, int NTH, int NSTR = 1>
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
        for (int q = 0; q < 8; ++q) v[q] = id[q] >= 0 ? w[(int64_t)id[q] * NSTR] : T(0);
        T s = v[0];
#pragma unroll
        for (int q = 1; q < 8; ++q) if (id[q] >= 0) s += v[q];
        for (int32_t q = 8; q < cnt; ++q) s += w[(int64_t)sh_idx[r.x + q] * NSTR];
        if (MASK && r.y < 0) s = T(0);
#pragma unroll
        for (int q = 0; q < 8; ++q) if (id[q] >= 0) w[(int64_t)id[q] * NSTR] = s;
        for (int32_t q = 8; q < cnt; ++q) w[(int64_t)sh_idx[r.x + q] * NSTR] = s;
    }
}

}  // namespace semgs
