// sem_fdm.cu — NEXT-2a: the fast-diagonalisation local solve of the Schwarz smoothers, Eq. (3).
// "The Schwarz smoothers are implemented by solving local Poisson problems on domains extended into adjacent
// elements by one layer.  Thus, for an 8 x 8 x 8 brick (N = 7), one solves a 10 x 10 x 10 local problem ... using fast
// diagonalization (FDM),   u^e = (S_z x S_y x S_x) Lambda^-1 (S_z^T x S_y^T x S_x^T) b^e,   e = 1..E,   where each 1D
// matrix of eigenvectors, S_*, is 10 x 10, and Lambda is a diagonal matrix with only 1,000 nonzeros.  The leading
// complexity is ~ 12 x 10^4 operations for the application of S_* and S_*^T (implemented as dgemm), with ~ 2,000 loads
// per element (for b^e and Lambda)."  Table 2/3: `fusedFDM`, the most expensive elliptic kernel (9.5 %).
//
// Kernel: 12 m^4 flops on (3 m^3 + 3 m^2) values per element = 9 flop/B in FP32 at m = 10: between the HBM roofline and
// the FP32 pipe, and -- as the paper found -- bound by shared-memory wavefronts if every product reads an operand from
// shared memory.  So the six 1-D contractions run in REGISTERS: a thread owns LPT whole lines of the m^3 block
// (m values along the contracted direction each), the rows of S_d are broadcast from shared memory with 128-bit loads
// and shared by the thread's lines, and between directions the block is re-distributed through shared memory once
// (line ownership rotates k-lines -> j-lines -> i-lines and back).  S_x^T, Lambda^-1 and S_x are applied by the same
// owner back to back, so there are 5 phases and 4 barriers; b is read and u written straight from/to registers with
// coalesced accesses.  This is not the paper's kernel (OCCA, one thread block per element, operands in shared memory).
#include "sem_internal.h"

namespace {

template <typename T> struct vec16;
template <> struct vec16<float> { using type = float4; static constexpr int n = 4; };
template <> struct vec16<double> { using type = double2; static constexpr int n = 2; };

template <typename T, int M>
struct fdm_cfg {
    static constexpr int VEC = vec16<T>::n;
    static constexpr int MP = (M + VEC - 1) / VEC * VEC;          // padded row length: rows start 16-byte aligned
    static constexpr int LINES = M * M;                           // lines per element and phase
    static constexpr int LPT = M >= 6 ? 2 : 1;                    // lines per thread (share every S row load)
    static constexpr int TPE = (LINES + LPT - 1) / LPT;           // threads per element
    static constexpr int EPC = (224 / TPE) > 0 ? 224 / TPE : 1;   // elements per CTA
    static constexpr int NT = EPC * TPE;
    static constexpr int S_EL = 3 * M * MP;                       // padded S values per element
    static constexpr int B_EL = M * M * MP;                       // padded block values per element
    static constexpr size_t SMEM = sizeof(T) * (size_t)EPC * (S_EL + B_EL);
};

// row[0..M) <- the M values at `src` (16-byte aligned, padded to MP), 128-bit shared-memory loads
template <typename T, int M>
__device__ __forceinline__ void load_row(const T* __restrict__ src, T (&row)[fdm_cfg<T, M>::MP]) {
    using V = typename vec16<T>::type;
    constexpr int VEC = vec16<T>::n;
#pragma unroll
    for (int q = 0; q < fdm_cfg<T, M>::MP / VEC; ++q) {
        const V v = reinterpret_cast<const V*>(src)[q];
        if constexpr (VEC == 4) {
            row[4 * q] = v.x; row[4 * q + 1] = v.y; row[4 * q + 2] = v.z; row[4 * q + 3] = v.w;
        } else {
            row[2 * q] = v.x; row[2 * q + 1] = v.y;
        }
    }
}

// out[r][o] = sum_l S[l][o] in[r][l]  (TRANSPOSED: S^T applied)   or   sum_l S[o][l] in[r][l]  (S applied);
// both walk the rows of S (sS: [M][MP]), each row loaded once for the thread's LPT lines.
template <typename T, int M, int LPT, bool TRANSPOSED>
__device__ __forceinline__ void contract_lines(const T* __restrict__ sS, const T (&in)[LPT][M], T (&out)[LPT][M]) {
    constexpr int MP = fdm_cfg<T, M>::MP;
    if constexpr (TRANSPOSED) {
#pragma unroll
        for (int r = 0; r < LPT; ++r)
#pragma unroll
            for (int o = 0; o < M; ++o) out[r][o] = T(0);
#pragma unroll
        for (int l = 0; l < M; ++l) {
            T row[MP];
            load_row<T, M>(sS + l * MP, row);
#pragma unroll
            for (int r = 0; r < LPT; ++r)
#pragma unroll
                for (int o = 0; o < M; ++o) out[r][o] += row[o] * in[r][l];
        }
    } else {
#pragma unroll
        for (int o = 0; o < M; ++o) {
            T row[MP];
            load_row<T, M>(sS + o * MP, row);
#pragma unroll
            for (int r = 0; r < LPT; ++r) {
                T s = T(0);
#pragma unroll
                for (int l = 0; l < M; ++l) s += row[l] * in[r][l];
                out[r][o] = s;
            }
        }
    }
}

template <typename T, int M>
__global__ void __launch_bounds__(fdm_cfg<T, M>::NT)
k_fdm(int64_t E, const T* __restrict__ S, const T* __restrict__ invL, const T* b, T* u) {
    using C = fdm_cfg<T, M>;
    constexpr int MP = C::MP, LPT = C::LPT, TPE = C::TPE, EPC = C::EPC, M2 = M * M, M3 = M * M * M;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sS_all = reinterpret_cast<T*>(smem_raw);
    T* sB_all = sS_all + EPC * C::S_EL;
    const int el = threadIdx.x / TPE, tl = threadIdx.x - el * TPE;
    T* sS = sS_all + el * C::S_EL;                       // [3][M][MP]: x, y, z
    T* sB = sB_all + el * C::B_EL;                       // [k][j][MP]
    const int64_t ngrp = (E + EPC - 1) / EPC;

    for (int64_t grp = blockIdx.x; grp < ngrp; grp += gridDim.x) {
        const int64_t e0 = grp * EPC, e = e0 + el;
        const bool live = e < E;
        const int ne = (int)((E - e0) < EPC ? (E - e0) : EPC);
        // ---- phase 1: owner (j,i) of a k-line: b from global, S_z^T in registers ----
        T in[LPT][M], out[LPT][M];
#pragma unroll
        for (int r = 0; r < LPT; ++r) {
            const int q = tl + r * TPE;
#pragma unroll
            for (int k = 0; k < M; ++k) in[r][k] = (live && q < M2) ? b[e * M3 + k * M2 + q] : T(0);
        }
        __syncthreads();                                 // previous group's phase 5 has finished reading sS
        for (int t = threadIdx.x; t < ne * 3 * M2; t += C::NT) {        // S of this group, rows padded to MP
            const int row = t / M, col = t - row * M;
            sS_all[row * MP + col] = S[e0 * 3 * M2 + t];
        }
        __syncthreads();
        contract_lines<T, M, LPT, true>(sS + 2 * M * MP, in, out);
#pragma unroll
        for (int r = 0; r < LPT; ++r) {
            const int q = tl + r * TPE;
            if (q < M2) {
                const int j = q / M, i = q - j * M;
#pragma unroll
                for (int k = 0; k < M; ++k) sB[(k * M + j) * MP + i] = out[r][k];
            }
        }
        __syncthreads();
        // ---- phase 2: owner (k,i) of a j-line: S_y^T ----
#pragma unroll
        for (int r = 0; r < LPT; ++r) {
            const int q = tl + r * TPE, k = q / M, i = q - k * M;
#pragma unroll
            for (int j = 0; j < M; ++j) in[r][j] = q < M2 ? sB[(k * M + j) * MP + i] : T(0);
        }
        contract_lines<T, M, LPT, true>(sS + M * MP, in, out);
#pragma unroll
        for (int r = 0; r < LPT; ++r) {                  // a j-line is read and written by its owner only: no barrier
            const int q = tl + r * TPE, k = q / M, i = q - k * M;
            if (q < M2)
#pragma unroll
                for (int j = 0; j < M; ++j) sB[(k * M + j) * MP + i] = out[r][j];
        }
        __syncthreads();
        // ---- phase 3: owner (k,j) of an i-line: S_x^T, Lambda^-1, S_x ----
        T il[LPT][M];
#pragma unroll
        for (int r = 0; r < LPT; ++r) {
            const int q = tl + r * TPE;
#pragma unroll
            for (int i = 0; i < M; ++i) il[r][i] = (live && q < M2) ? invL[e * M3 + q * M + i] : T(0);
        }
#pragma unroll
        for (int r = 0; r < LPT; ++r) {
            const int q = tl + r * TPE;
            T row[MP];
            if (q < M2) load_row<T, M>(sB + q * MP, row);
#pragma unroll
            for (int i = 0; i < M; ++i) in[r][i] = q < M2 ? row[i] : T(0);
        }
        contract_lines<T, M, LPT, true>(sS, in, out);
#pragma unroll
        for (int r = 0; r < LPT; ++r)
#pragma unroll
            for (int i = 0; i < M; ++i) out[r][i] *= il[r][i];
        contract_lines<T, M, LPT, false>(sS, out, in);
#pragma unroll
        for (int r = 0; r < LPT; ++r) {
            const int q = tl + r * TPE;
            if (q < M2)
#pragma unroll
                for (int i = 0; i < M; ++i) sB[q * MP + i] = in[r][i];
        }
        __syncthreads();
        // ---- phase 4: owner (k,i) of a j-line: S_y ----
#pragma unroll
        for (int r = 0; r < LPT; ++r) {
            const int q = tl + r * TPE, k = q / M, i = q - k * M;
#pragma unroll
            for (int j = 0; j < M; ++j) in[r][j] = q < M2 ? sB[(k * M + j) * MP + i] : T(0);
        }
        contract_lines<T, M, LPT, false>(sS + M * MP, in, out);
#pragma unroll
        for (int r = 0; r < LPT; ++r) {
            const int q = tl + r * TPE, k = q / M, i = q - k * M;
            if (q < M2)
#pragma unroll
                for (int j = 0; j < M; ++j) sB[(k * M + j) * MP + i] = out[r][j];
        }
        __syncthreads();
        // ---- phase 5: owner (j,i) of a k-line: S_z, u to global ----
#pragma unroll
        for (int r = 0; r < LPT; ++r) {
            const int q = tl + r * TPE, j = q / M, i = q - j * M;
#pragma unroll
            for (int k = 0; k < M; ++k) in[r][k] = q < M2 ? sB[(k * M + j) * MP + i] : T(0);
        }
        contract_lines<T, M, LPT, false>(sS + 2 * M * MP, in, out);
#pragma unroll
        for (int r = 0; r < LPT; ++r) {
            const int q = tl + r * TPE;
            if (live && q < M2)
#pragma unroll
                for (int k = 0; k < M; ++k) u[e * M3 + k * M2 + q] = out[r][k];
        }
    }
}

template <typename T, int M>
int launch_m(sem_ctx* c, const void* S, const void* invL, const void* b, void* u) {
    using C = fdm_cfg<T, M>;
    static int resident = 0;                             // CTAs per SM of this instantiation
    auto kern = k_fdm<T, M>;
    if (!resident) {
        if (C::SMEM > 48 * 1024)
            SEM_CUDA_OK(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
        int nb = 0;
        SEM_CUDA_OK(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, C::NT, C::SMEM));
        resident = nb > 0 ? nb : 1;
    }
    const int64_t ngrp = (c->E + C::EPC - 1) / C::EPC;
    int64_t grid = (int64_t)c->num_sms * resident;       // single wave of persistent CTAs
    if (grid > ngrp) grid = ngrp;
    kern<<<(unsigned)grid, C::NT, C::SMEM, c->stream>>>(c->E, (const T*)S, (const T*)invL, (const T*)b, (T*)u);
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

template <typename T>
int launch(sem_ctx* c, int m, const void* S, const void* invL, const void* b, void* u) {
    switch (m) {
#define SEM_FDM_CASE(MM) case MM: return launch_m<T, MM>(c, S, invL, b, u);
        SEM_FDM_CASE(2) SEM_FDM_CASE(3) SEM_FDM_CASE(4) SEM_FDM_CASE(5) SEM_FDM_CASE(6) SEM_FDM_CASE(7) SEM_FDM_CASE(8)
        SEM_FDM_CASE(9) SEM_FDM_CASE(10) SEM_FDM_CASE(11) SEM_FDM_CASE(12) SEM_FDM_CASE(13) SEM_FDM_CASE(14)
        SEM_FDM_CASE(15) SEM_FDM_CASE(16)
#undef SEM_FDM_CASE
    }
    return sem_fail(c, SEM_EINVAL, "sem_fdm_apply: m = %d outside 2..16", m);
}

}  // namespace

extern "C" int sem_fdm_apply(sem_ctx* ctx, int m, const void* S, const void* inv_lambda, const void* b, void* u,
                             sem_prec prec) {
    if (!ctx) return SEM_EINVAL;
    ctx->err.clear();
    if (!S || !inv_lambda || !b || !u) return sem_fail(ctx, SEM_EINVAL, "sem_fdm_apply: NULL pointer");
    if (prec != SEM_F64 && prec != SEM_F32) return sem_fail(ctx, SEM_EINVAL, "sem_fdm_apply: bad sem_prec");
    if (m < 2 || m > 16) return sem_fail(ctx, SEM_EINVAL, "sem_fdm_apply: m = %d outside 2..16", m);
    if (prec == SEM_F64) return launch<double>(ctx, m, S, inv_lambda, b, u);
    return launch<float>(ctx, m, S, inv_lambda, b, u);
}
