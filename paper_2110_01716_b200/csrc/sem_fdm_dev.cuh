// sem_fdm_dev.cuh -- the kernel of sem_fdm.cu (design notes there).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

namespace sem_fdm_dev {


template <typename T> struct vec16;
template <> struct vec16<float> { using type = float4; static constexpr int n = 4; };
template <> struct vec16<double> { using type = double2; static constexpr int n = 2; };

// LPT_ = lines per thread (they share every S row load), EPC_ = elements per CTA
template <typename T, int M, int LPT_, int EPC_>
struct fdm_cfg {
    static constexpr int VEC = vec16<T>::n;
    static constexpr int MP = (M + VEC - 1) / VEC * VEC;          // padded row length: rows start 16-byte aligned
    static constexpr int LINES = M * M;                           // lines per element and phase
    static constexpr int LPT = LPT_;
    static constexpr int TPE = (LINES + LPT - 1) / LPT;           // threads per element
    static constexpr int EPC = EPC_;
    static constexpr int NT = EPC * TPE;
    static constexpr int S_EL = 3 * M * MP;                       // padded S values per element
    // plane stride of the block: the lanes of a warp that own j-lines span several k-planes; their bank ranges
    // [0, M) + k * PS must not overlap, so PS = MP modulo one bank cycle (32 floats / 16 doubles), rows stay 16-byte aligned
    static constexpr int BANKW = 128 / (int)sizeof(T);
    static constexpr int PS = M * MP + ((MP - M * MP) % BANKW + BANKW) % BANKW;
    static constexpr int B_EL = M * PS;                           // padded block values per element
    static constexpr int STAGE = EPC * (S_EL + 2 * B_EL);         // S, Lambda^-1 and the block of EPC elements
    static constexpr size_t SMEM1 = sizeof(T) * (size_t)STAGE;    // per stage
};

// row[0..M) <- the M values at `src` (16-byte aligned, padded to MP), 128-bit shared-memory loads
template <typename T, int M>
__device__ __forceinline__ void load_row(const T* __restrict__ src, T (&row)[fdm_cfg<T, M, 1, 1>::MP]) {
    using V = typename vec16<T>::type;
    constexpr int VEC = vec16<T>::n;
#pragma unroll
    for (int q = 0; q < fdm_cfg<T, M, 1, 1>::MP / VEC; ++q) {
        const V v = reinterpret_cast<const V*>(src)[q];
        if constexpr (VEC == 4) {
            row[4 * q] = v.x; row[4 * q + 1] = v.y; row[4 * q + 2] = v.z; row[4 * q + 3] = v.w;
        } else {
            row[2 * q] = v.x; row[2 * q + 1] = v.y;
        }
    }
}

// One 1-D contraction of the thread's LPT lines, walking the rows of S (sS: [M][MP]) so that each row is loaded once
// for all of them.  ld(r, l) yields element l of line r, st(r, o, v) takes element o of the result.
//   TRANSPOSED (S^T applied):  out[o] = sum_l S[l][o] in[l]: the inputs are consumed one at a time (read just in time,
//                              never all live), the M accumulators per line stay in registers and are stored at the end;
//   otherwise  (S applied):    out[o] = sum_l S[o][l] in[l]: the inputs are read first, every result is stored as soon as
//                              its dot product is done (never all live).
// Either way a line costs M + small registers instead of 2 M.
template <typename T, int M, int LPT, bool TRANSPOSED, class Ld, class St>
__device__ __forceinline__ void contract_lines(const T* __restrict__ sS, Ld ld, St st) {
    constexpr int MP = fdm_cfg<T, M, 1, 1>::MP;
    if constexpr (TRANSPOSED) {
        T acc[LPT][M];
#pragma unroll
        for (int r = 0; r < LPT; ++r)
#pragma unroll
            for (int o = 0; o < M; ++o) acc[r][o] = T(0);
#pragma unroll
        for (int l = 0; l < M; ++l) {
            T row[MP];
            load_row<T, M>(sS + l * MP, row);
#pragma unroll
            for (int r = 0; r < LPT; ++r) {
                const T v = ld(r, l);
#pragma unroll
                for (int o = 0; o < M; ++o) acc[r][o] += row[o] * v;
            }
        }
#pragma unroll
        for (int r = 0; r < LPT; ++r)
#pragma unroll
            for (int o = 0; o < M; ++o) st(r, o, acc[r][o]);
    } else {
        T in[LPT][M];
#pragma unroll
        for (int r = 0; r < LPT; ++r)
#pragma unroll
            for (int l = 0; l < M; ++l) in[r][l] = ld(r, l);
#pragma unroll
        for (int o = 0; o < M; ++o) {
            T row[MP];
            load_row<T, M>(sS + o * MP, row);
#pragma unroll
            for (int r = 0; r < LPT; ++r) {
                T v = T(0);
#pragma unroll
                for (int l = 0; l < M; ++l) v += row[l] * in[r][l];
                st(r, o, v);
            }
        }
    }
}

// cp.async (LDGSTS) of BYTES (4, 8 or 16) from global to shared memory, no registers in between
template <int BYTES>
__device__ __forceinline__ void cp_async(void* smem_dst, const void* gsrc) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(d), "l"(gsrc), "n"(BYTES) : "memory");
}

// rows of M values, contiguous in global memory, to rows padded to MP in shared memory, by all NT threads of the CTA
// (PS = stride of a plane of M rows in shared memory)
template <typename T, int M, int NT, int PS>
__device__ __forceinline__ void copy_rows_async(T* __restrict__ sdst, const T* __restrict__ gsrc, int nrows) {
    constexpr int MP = fdm_cfg<T, M, 1, 1>::MP;
    constexpr int RB = M * (int)sizeof(T);
    constexpr int CH = RB % 16 == 0 ? 16 : RB % 8 == 0 ? 8 : 4;      // chunk bytes: row starts stay CH-aligned
    constexpr int CPR = RB / CH, VPC = CH / (int)sizeof(T);
    for (int t = threadIdx.x; t < nrows * CPR; t += NT) {
        const int row = t / CPR, c = t - row * CPR;
        const int plane = row / M;
        cp_async<CH>(sdst + plane * PS + (row - plane * M) * MP + c * VPC, gsrc + (int64_t)row * M + c * VPC);
    }
}

// Where the m^3 blocks come from and where the result goes.
//   PlainIO    b[E][m^3] -> u[E][m^3] (sem_fdm_apply).
//   SchwarzIO  the restricted additive Schwarz smoother in ONE kernel (NEXT-2b, sem_schwarz.cu): the block is GATHERED
//              from the residual r -- the element's own nodes into the interior, the face neighbours' one-layer-in
//              values into the 6 face layers through the links resolved at setup, zeros on the block's edges and corners
//              -- by 4/8-byte cp.async straight into shared memory, and only the element's own part of the solution
//              is written, weighted (W = 1 / multiplicity): the blocks never touch HBM.
template <typename T, int M>
struct PlainIO {
    const T* b;
    T* u;
    static constexpr size_t extra_bytes(int) { return 0; }
    template <int NT, int PS>
    __device__ __forceinline__ void load(T* __restrict__ sB, unsigned char*, int64_t e0, int ne) const {
        copy_rows_async<T, M, NT, PS>(sB, b + e0 * (M * M * M), ne * M * M);
    }
    __device__ __forceinline__ void store(const unsigned char*, int, int64_t e, int o, int q, T v) const {
        u[e * (M * M * M) + o * (M * M) + q] = v;
    }
};

template <typename T, int M>
struct SchwarzIO {
    const T* r;            // residual, local layout [E][p^3], p = M - 2
    const int4* link;      // [E][6] (neighbour, base, stride a, stride b), neighbour < 0: none
    const int32_t* nrm;    // [E][6] neighbour's face axis | side << 2
    const T* W;            // [E][p^3] weight of the result
    T* z;                  // [E][p^3]
    // per element of the CTA, after the stage(s): the 6 links (int4 + int) and the element's weights (cp.async too)
    static constexpr int P = M - 2, P3 = P * P * P;
    static constexpr size_t EL_BYTES = 128 + ((P3 * sizeof(T) + 15) / 16) * 16;
    static constexpr size_t extra_bytes(int epc) { return (size_t)epc * EL_BYTES; }
    template <int NT, int PS>
    __device__ __forceinline__ void load(T* __restrict__ sB0, unsigned char* extra, int64_t e0, int ne) const {
        constexpr int P2 = P * P, MP = fdm_cfg<T, M, 1, 1>::MP, B_EL = M * PS;
        for (int t = threadIdx.x; t < ne * 6; t += NT) {                               // links of the group, once
            const int el = t / 6, f = t - el * 6;
            int4* lk = reinterpret_cast<int4*>(extra + el * EL_BYTES);
            int32_t* nf = reinterpret_cast<int32_t*>(extra + el * EL_BYTES + 96);
            lk[f] = link[(e0 + el) * 6 + f];
            nf[f] = nrm[(e0 + el) * 6 + f];
        }
        __syncthreads();
        for (int el = 0; el < ne; ++el) {
            const int64_t e = e0 + el;
            T* sB = sB0 + el * B_EL;
            const int4* lk6 = reinterpret_cast<const int4*>(extra + el * EL_BYTES);
            const int32_t* nf6 = reinterpret_cast<const int32_t*>(extra + el * EL_BYTES + 96);
            T* sW = reinterpret_cast<T*>(extra + el * EL_BYTES + 128);
            for (int t = threadIdx.x; t < P3; t += NT) {                               // own nodes, and their weights
                const int i = t % P, j = (t / P) % P, k = t / P2;
                cp_async<(int)sizeof(T)>(sB + (k + 1) * PS + (j + 1) * MP + (i + 1), r + e * P3 + t);
                cp_async<(int)sizeof(T)>(sW + t, W + e * P3 + t);
            }
            for (int t = threadIdx.x; t < 6 * P2; t += NT) {                           // face layers
                const int f = t / P2, fa = (t % P2) % P, fb = (t % P2) / P, axis = f >> 1, g = (f & 1) ? M - 1 : 0;
                const int a = axis == 0 ? g : fa + 1, b = axis == 0 ? fa + 1 : (axis == 1 ? g : fb + 1),
                          c = axis == 2 ? g : fb + 1;
                const int4 lk = lk6[f];
                T* dst = sB + c * PS + b * MP + a;
                if (lk.x >= 0) {
                    const int nf = nf6[f], na = nf & 3, ns = nf >> 2;
                    const int stride = na == 0 ? 1 : (na == 1 ? P : P2);
                    const int l = lk.y + fa * lk.z + fb * lk.w + (ns ? -stride : stride);
                    cp_async<(int)sizeof(T)>(dst, r + (int64_t)lk.x * P3 + l);
                } else {
                    *dst = T(0);
                }
            }
            for (int t = threadIdx.x; t < 12 * P + 8; t += NT) {                       // edges and corners: no node
                int a, b, c;
                if (t < 12 * P) {
                    const int ed = t / P, q = t % P + 1, ax = ed >> 2, s0 = (ed & 1) ? M - 1 : 0, s1 = (ed & 2) ? M - 1 : 0;
                    a = ax == 0 ? q : s0;
                    b = ax == 1 ? q : (ax == 0 ? s0 : s1);
                    c = ax == 2 ? q : s1;
                } else {
                    const int cn = t - 12 * P;
                    a = (cn & 1) ? M - 1 : 0; b = (cn & 2) ? M - 1 : 0; c = (cn & 4) ? M - 1 : 0;
                }
                sB[c * PS + b * MP + a] = T(0);
            }
        }
    }
    __device__ __forceinline__ void store(const unsigned char* extra, int el, int64_t e, int o, int q, T v) const {
        const int j = q / M, i = q - j * M;
        if (o >= 1 && o <= P && j >= 1 && j <= P && i >= 1 && i <= P) {
            const int l = ((o - 1) * P + (j - 1)) * P + (i - 1);
            const T* sW = reinterpret_cast<const T*>(extra + el * EL_BYTES + 128);
            z[e * P3 + l] = sW[l] * v;
        }
    }
};

// MINB = resident CTAs per SM the register allocation is held to.  NSTAGE = 2: two shared-memory stages of
// {S, Lambda^-1, block}: while a group of EPC elements is worked on in one stage, the next group's operands land in the
// other (cp.async).  NSTAGE = 1: one stage (half the shared memory, twice the resident CTAs hide the copy instead).
template <typename T, int M, int LPT_, int EPC_, int MINB, int NSTAGE, class IO = PlainIO<T, M>>
__global__ void __launch_bounds__((fdm_cfg<T, M, LPT_, EPC_>::NT), MINB)
k_fdm(int64_t E, const T* __restrict__ S, const T* __restrict__ invL, const IO io) {
    using C = fdm_cfg<T, M, LPT_, EPC_>;
    constexpr int MP = C::MP, LPT = C::LPT, TPE = C::TPE, EPC = C::EPC, M2 = M * M, M3 = M * M * M, NT = C::NT;
    constexpr int STG = C::STAGE, PS = C::PS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* smem = reinterpret_cast<T*>(smem_raw);
    unsigned char* xtra = smem_raw + sizeof(T) * (size_t)(NSTAGE * STG);     // the I/O policy's own area (one stage only)
    const int el = threadIdx.x / TPE, tl = threadIdx.x - el * TPE;
    const int64_t ngrp = (E + EPC - 1) / EPC;

    auto issue = [&](int64_t grp, int stage) {
        const int64_t e0 = grp * EPC;
        const int ne = (int)((E - e0) < EPC ? (E - e0) : EPC);
        T* st = smem + stage * STG;
        copy_rows_async<T, M, NT, M * MP>(st, S + e0 * 3 * M2, ne * 3 * M);
        copy_rows_async<T, M, NT, PS>(st + EPC * C::S_EL, invL + e0 * M3, ne * M2);
        io.template load<NT, PS>(st + EPC * (C::S_EL + C::B_EL), xtra, e0, ne);
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    if (NSTAGE == 2 && (int64_t)blockIdx.x < ngrp) issue(blockIdx.x, 0);
    int stage = 0;
    for (int64_t grp = blockIdx.x; grp < ngrp; grp += gridDim.x, stage ^= (NSTAGE - 1)) {
        const int64_t e = grp * EPC + el;
        const bool live = e < E;
        T* stg = smem + stage * STG;
        const T* sS = stg + el * C::S_EL;                              // [3][M][MP]: x, y, z
        const T* sL = stg + EPC * C::S_EL + el * C::B_EL;              // [c][b][MP]
        T* sB = stg + EPC * (C::S_EL + C::B_EL) + el * C::B_EL;        // [k][j][MP]
        if (NSTAGE == 1) {
            __syncthreads();              // the previous group is no longer read
            issue(grp, 0);
        }
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();                  // this stage has landed for everyone; the other stage is no longer read
        if (NSTAGE == 2 && grp + gridDim.x < ngrp) issue(grp + gridDim.x, stage ^ 1);
        int q[LPT], a[LPT], c[LPT];       // line q = a * M + c of the element
        bool ok[LPT];
#pragma unroll
        for (int r = 0; r < LPT; ++r) {
            q[r] = tl + r * TPE;
            ok[r] = q[r] < M2;
            if (!ok[r]) q[r] = M2 - 1;                // an idle slot (M^2 not a multiple of LPT) computes but never stores
            a[r] = q[r] / M;
            c[r] = q[r] - a[r] * M;
        }
        // line ownership: "outer" = (j,i) owns a k-line (element l at (l*M + a)*MP + c); "mid" = (k,i) owns a j-line
        // (element l at (a*M + l)*MP + c); "inner" = (k,j) owns an i-line (row q).  A line is read and written by its
        // owner only, so the barriers sit between the phases and nowhere else.
        auto ld_outer = [&](int r, int l) { return sB[l * PS + a[r] * MP + c[r]]; };
        auto st_outer = [&](int r, int o, T v) { if (ok[r]) sB[o * PS + a[r] * MP + c[r]] = v; };
        auto ld_mid = [&](int r, int l) { return sB[a[r] * PS + l * MP + c[r]]; };
        auto st_mid = [&](int r, int o, T v) { if (ok[r]) sB[a[r] * PS + o * MP + c[r]] = v; };
        // ---- phase 1: S_z^T on k-lines ----
        contract_lines<T, M, LPT, true>(sS + 2 * M * MP, ld_outer, st_outer);
        __syncthreads();
        // ---- phase 2: S_y^T on j-lines ----
        contract_lines<T, M, LPT, true>(sS + M * MP, ld_mid, st_mid);
        __syncthreads();
        // ---- phase 3: S_x^T, Lambda^-1, S_x on i-lines (rows: 128-bit accesses) ----
        {
            T v[LPT][MP];
#pragma unroll
            for (int r = 0; r < LPT; ++r) load_row<T, M>(sB + a[r] * PS + c[r] * MP, v[r]);
            T w[LPT][M];
            contract_lines<T, M, LPT, true>(sS, [&](int r, int l) { return v[r][l]; },
                                            [&](int r, int o, T x) { w[r][o] = x; });
#pragma unroll
            for (int r = 0; r < LPT; ++r) {
                load_row<T, M>(sL + a[r] * PS + c[r] * MP, v[r]);
#pragma unroll
                for (int i = 0; i < M; ++i) w[r][i] *= v[r][i];
            }
            contract_lines<T, M, LPT, false>(sS, [&](int r, int l) { return w[r][l]; },
                                             [&](int r, int o, T x) { if (ok[r]) sB[a[r] * PS + c[r] * MP + o] = x; });
        }
        __syncthreads();
        // ---- phase 4: S_y on j-lines ----
        contract_lines<T, M, LPT, false>(sS + M * MP, ld_mid, st_mid);
        __syncthreads();
        // ---- phase 5: S_z on k-lines, u to global (coalesced) ----
        contract_lines<T, M, LPT, false>(sS + 2 * M * MP, ld_outer, [&](int r, int o, T x) {
            if (live && ok[r]) io.store(xtra, el, e, o, q[r], x);
        });
    }
}

// ---- variant with S_d resident in registers ------------------------------------------------------------------------
// k_fdm above reads every row of S_d from shared memory once per LPT lines, and a warp-uniform 128-bit load still costs
// two shared-memory wavefronts: those broadcasts are 55 % of its wavefronts, and the shared-memory pipe is its limiter.
// Here a thread loads the whole m x m matrix of the phase into registers ONCE and then walks its LPS lines one after the
// other (a line needs m inputs and one running dot product, so the lines do not multiply the register count):
// m^2 / 4 broadcast loads per thread and phase instead of (m^2 / 4) x LPS / LPT.  Phase 3 uses the same S_x registers for
// S_x^T and S_x.  FP32 up to m = 12 and FP64 up to m = 8 fit the register file.
template <typename T, int M>
__device__ __forceinline__ void load_matrix(const T* __restrict__ sS, T (&Sr)[M][fdm_cfg<T, M, 1, 1>::MP]) {
#pragma unroll
    for (int l = 0; l < M; ++l) load_row<T, M>(sS + l * fdm_cfg<T, M, 1, 1>::MP, Sr[l]);
}

// out[o] = sum_l (TRANSPOSED ? S[l][o] : S[o][l]) in[l], each result handed to st as soon as it is complete
template <typename T, int M, bool TRANSPOSED, class St>
__device__ __forceinline__ void apply_matrix(const T (&Sr)[M][fdm_cfg<T, M, 1, 1>::MP], const T (&in)[M], St st) {
#pragma unroll
    for (int o = 0; o < M; ++o) {
        T v = T(0);
#pragma unroll
        for (int l = 0; l < M; ++l) v += (TRANSPOSED ? Sr[l][o] : Sr[o][l]) * in[l];
        st(o, v);
    }
}

template <typename T, int M, int LPS, int EPC_, int MINB, int NSTAGE, class IO = PlainIO<T, M>>
__global__ void __launch_bounds__((fdm_cfg<T, M, LPS, EPC_>::NT), MINB)
k_fdm_sreg(int64_t E, const T* __restrict__ S, const T* __restrict__ invL, const IO io) {
    using C = fdm_cfg<T, M, LPS, EPC_>;
    constexpr int MP = C::MP, TPE = C::TPE, EPC = C::EPC, M2 = M * M, M3 = M * M * M, NT = C::NT;
    constexpr int STG = C::STAGE, PS = C::PS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* smem = reinterpret_cast<T*>(smem_raw);
    unsigned char* xtra = smem_raw + sizeof(T) * (size_t)(NSTAGE * STG);     // the I/O policy's own area (one stage only)
    const int el = threadIdx.x / TPE, tl = threadIdx.x - el * TPE;
    const int64_t ngrp = (E + EPC - 1) / EPC;

    auto issue = [&](int64_t grp, int stage) {
        const int64_t e0 = grp * EPC;
        const int ne = (int)((E - e0) < EPC ? (E - e0) : EPC);
        T* st = smem + stage * STG;
        copy_rows_async<T, M, NT, M * MP>(st, S + e0 * 3 * M2, ne * 3 * M);
        copy_rows_async<T, M, NT, PS>(st + EPC * C::S_EL, invL + e0 * M3, ne * M2);
        io.template load<NT, PS>(st + EPC * (C::S_EL + C::B_EL), xtra, e0, ne);
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    if (NSTAGE == 2 && (int64_t)blockIdx.x < ngrp) issue(blockIdx.x, 0);
    int stage = 0;
    for (int64_t grp = blockIdx.x; grp < ngrp; grp += gridDim.x, stage ^= (NSTAGE - 1)) {
        const int64_t e = grp * EPC + el;
        const bool live = e < E;
        T* stg = smem + stage * STG;
        const T* sS = stg + el * C::S_EL;                              // [3][M][MP]: x, y, z
        const T* sL = stg + EPC * C::S_EL + el * C::B_EL;              // [c][b][MP]
        T* sB = stg + EPC * (C::S_EL + C::B_EL) + el * C::B_EL;        // [k][j][MP]
        if (NSTAGE == 1) {
            __syncthreads();
            issue(grp, 0);
        }
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();
        if (NSTAGE == 2 && grp + gridDim.x < ngrp) issue(grp + gridDim.x, stage ^ 1);
        T Sr[M][MP];
        // One phase over the thread's lines q = tl, tl + TPE, ...: line element l sits at base(q) + l * STRIDE.
        // OUTER: q = (j,i), k-line;  MID: q = (k,i), j-line.  In place: a line is read whole before it is written.
        auto phase = [&](auto transposed, auto outer) {
            constexpr bool TR = decltype(transposed)::value, OUTER = decltype(outer)::value;
            constexpr int STRIDE = OUTER ? PS : MP;
#pragma unroll 1
            for (int q = tl; q < M2; q += TPE) {
                const int a = q / M, c = q - a * M;
                T* line = sB + (OUTER ? a * MP + c : a * PS + c);
                T in[M];
#pragma unroll
                for (int l = 0; l < M; ++l) in[l] = line[l * STRIDE];
                apply_matrix<T, M, TR>(Sr, in, [&](int o, T v) { line[o * STRIDE] = v; });
            }
        };
        // ---- phase 1: S_z^T on k-lines ----
        load_matrix<T, M>(sS + 2 * M * MP, Sr);
        phase(std::true_type{}, std::true_type{});
        __syncthreads();
        // ---- phase 2: S_y^T on j-lines ----
        load_matrix<T, M>(sS + M * MP, Sr);
        phase(std::true_type{}, std::false_type{});
        __syncthreads();
        // ---- phase 3: S_x^T, Lambda^-1, S_x on i-lines (rows: 128-bit accesses) ----
        load_matrix<T, M>(sS, Sr);
#pragma unroll 1
        for (int q = tl; q < M2; q += TPE) {
            T row[MP], il[MP], t[M];
            const int a = q / M, ro = a * PS + (q - a * M) * MP;
            load_row<T, M>(sB + ro, row);
            load_row<T, M>(sL + ro, il);
            T in[M];
#pragma unroll
            for (int l = 0; l < M; ++l) in[l] = row[l];
            apply_matrix<T, M, true>(Sr, in, [&](int o, T v) { t[o] = v * il[o]; });
            apply_matrix<T, M, false>(Sr, t, [&](int o, T v) { sB[ro + o] = v; });
        }
        __syncthreads();
        // ---- phase 4: S_y on j-lines ----
        load_matrix<T, M>(sS + M * MP, Sr);
        phase(std::false_type{}, std::false_type{});
        __syncthreads();
        // ---- phase 5: S_z on k-lines, u to global (coalesced) ----
        load_matrix<T, M>(sS + 2 * M * MP, Sr);
#pragma unroll 1
        for (int q = tl; q < M2; q += TPE) {
            const int a = q / M, c = q - a * M;
            const T* line = sB + a * MP + c;
            T in[M];
#pragma unroll
            for (int l = 0; l < M; ++l) in[l] = line[l * PS];
            apply_matrix<T, M, false>(Sr, in, [&](int o, T v) {
                if (live) io.store(xtra, el, e, o, q, v);
            });
        }
    }
}

// ---- tensor-core variant (FP32): every 1-D contraction as mma.sync.m16n8k8 TF32 in three passes -----------------------
// P:107 "the application of S and S^T (implemented as dgemm)": a contraction of the m^2 lines of a block with an m x m
// matrix IS a small GEMM, [m^2 x m] x [m x m].  One warp per element; 16 lines form the M dimension of an MMA tile, the
// contraction index and the output index are padded to multiples of 8 (zeros), the matrix of the phase is the B operand
// (split once per phase into hi + lo TF32 parts, as in ax_tf32: hi*hi + lo*hi + hi*lo, FP32 accumulation, FP32-level
// accuracy).  A tile's lines are read by that tile only, so the block is updated in place with one __syncwarp per tile.
__device__ __forceinline__ void fdm_split_tf32(float x, uint32_t& hi, uint32_t& lo) {
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(hi) : "f"(x));
    const float rest = x - __uint_as_float(hi);
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(lo) : "f"(rest));
}
__device__ __forceinline__ void fdm_mma1688(float (&d)[4], const uint32_t (&a)[4], const uint32_t (&b)[2]) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}

// One phase: out[line][o] = sum_l Mat[o][l] in[line][l] for all M^2 lines of direction DIR (0: i-lines, 1: j-lines,
// 2: k-lines), Mat = S (TRANSPOSED: S^T), in place in the block sB.  SCALE: the result is multiplied by Lambda^-1 (sL, same
// layout as the block).  LAST: the result goes to the I/O policy instead of the block.
template <int M, int DIR, bool TRANSPOSED, bool SCALE, bool LAST, class IO>
__device__ __forceinline__ void fdm_mma_phase(float* __restrict__ sB, const float* __restrict__ sS,
                                              const float* __restrict__ sL, const IO& io, const unsigned char* xtra,
                                              int64_t e) {
    using C = fdm_cfg<float, M, 1, 1>;
    constexpr int MP = C::MP, PS = C::PS, M2 = M * M;
    constexpr int KS = (M + 7) / 8, NTI = (M + 7) / 8, TILES = (M2 + 15) / 16;
    constexpr int LSTR = DIR == 0 ? 1 : (DIR == 1 ? MP : PS);         // stride of the line's own index
    const int lane = threadIdx.x, g = lane >> 2, t = lane & 3;
    // B fragments of the phase: B[l][o] = Mat[o][l];  Mat = S^T: S[l][o], Mat = S: S[o][l];  S row-major [M][MP]
    uint32_t bh[KS][NTI][2], bl[KS][NTI][2];
#pragma unroll
    for (int ks = 0; ks < KS; ++ks)
#pragma unroll
        for (int nt = 0; nt < NTI; ++nt)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int l = ks * 8 + t + 4 * h, o = nt * 8 + g;
                const float v = (l < M && o < M) ? (TRANSPOSED ? sS[l * MP + o] : sS[o * MP + l]) : 0.f;
                fdm_split_tf32(v, bh[ks][nt][h], bl[ks][nt][h]);
            }
#pragma unroll 1
    for (int T = 0; T < TILES; ++T) {
        int base[2];
        bool ok[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int q = T * 16 + g + 8 * h;
            ok[h] = q < M2;
            const int a = ok[h] ? q / M : 0, c = ok[h] ? q - a * M : 0;
            base[h] = DIR == 0 ? a * PS + c * MP : (DIR == 1 ? a * PS + c : a * MP + c);
        }
        uint32_t ah[KS][4], al[KS][4];
#pragma unroll
        for (int ks = 0; ks < KS; ++ks)
#pragma unroll
            for (int f = 0; f < 4; ++f) {                               // a0 (g, t), a1 (g+8, t), a2 (g, t+4), a3 (g+8, t+4)
                const int h = f & 1, l = ks * 8 + t + 4 * (f >> 1);
                const float v = (ok[h] && l < M) ? sB[base[h] + l * LSTR] : 0.f;
                fdm_split_tf32(v, ah[ks][f], al[ks][f]);
            }
        float acc[NTI][4];
#pragma unroll
        for (int nt = 0; nt < NTI; ++nt) {
            acc[nt][0] = acc[nt][1] = acc[nt][2] = acc[nt][3] = 0.f;
#pragma unroll
            for (int ks = 0; ks < KS; ++ks) {
                fdm_mma1688(acc[nt], al[ks], bh[ks][nt]);
                fdm_mma1688(acc[nt], ah[ks], bl[ks][nt]);
                fdm_mma1688(acc[nt], ah[ks], bh[ks][nt]);
            }
        }
        __syncwarp();                                                   // every lane holds its inputs: the lines may be overwritten
#pragma unroll
        for (int nt = 0; nt < NTI; ++nt)
#pragma unroll
            for (int f = 0; f < 4; ++f) {                               // c0 (g, 2t), c1 (g, 2t+1), c2 (g+8, 2t), c3 (g+8, 2t+1)
                const int h = f >> 1, o = nt * 8 + 2 * t + (f & 1);
                if (!ok[h] || o >= M) continue;
                float v = acc[nt][f];
                if constexpr (SCALE) v *= sL[base[h] + o * LSTR];
                if constexpr (LAST) io.store(xtra, 0, e, o, T * 16 + g + 8 * h, v);      // DIR == 2: o = k, line = j * M + i
                else sB[base[h] + o * LSTR] = v;
            }
    }
    __syncwarp();
}

template <int M, int MINB, class IO>
__global__ void __launch_bounds__(32, MINB) k_fdm_mma(int64_t E, const float* __restrict__ S, const float* __restrict__ invL,
                                                      const IO io) {
    using C = fdm_cfg<float, M, 1, 1>;
    constexpr int MP = C::MP, PS = C::PS, M2 = M * M, M3 = M2 * M, NT = 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* smem = reinterpret_cast<float*>(smem_raw);
    unsigned char* xtra = smem_raw + sizeof(float) * (size_t)C::STAGE;
    float* sS = smem;                                   // [3][M][MP]: x, y, z
    float* sL = smem + C::S_EL;                         // [c][b][MP]
    float* sB = smem + C::S_EL + C::B_EL;               // [k][j][MP]
    for (int64_t e = blockIdx.x; e < E; e += gridDim.x) {
        __syncthreads();                                // the previous element is no longer read
        copy_rows_async<float, M, NT, M * MP>(sS, S + e * 3 * M2, 3 * M);
        copy_rows_async<float, M, NT, PS>(sL, invL + e * M3, M2);
        io.template load<NT, PS>(sB, xtra, e, 1);
        asm volatile("cp.async.commit_group;" ::: "memory");
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();
        fdm_mma_phase<M, 2, true, false, false>(sB, sS + 2 * M * MP, sL, io, xtra, e);     // S_z^T
        fdm_mma_phase<M, 1, true, false, false>(sB, sS + M * MP, sL, io, xtra, e);         // S_y^T
        fdm_mma_phase<M, 0, true, true, false>(sB, sS, sL, io, xtra, e);                   // S_x^T, then Lambda^-1
        fdm_mma_phase<M, 0, false, false, false>(sB, sS, sL, io, xtra, e);                 // S_x
        fdm_mma_phase<M, 1, false, false, false>(sB, sS + M * MP, sL, io, xtra, e);        // S_y
        fdm_mma_phase<M, 2, false, false, true>(sB, sS + 2 * M * MP, sL, io, xtra, e);     // S_z, result to the policy
    }
}

}  // namespace sem_fdm_dev
