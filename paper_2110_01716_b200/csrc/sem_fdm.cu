// sem_fdm.cu — NEXT-2a: the fast-diagonalisation local solve of the Schwarz smoothers, Eq. (3).
// "The Schwarz smoothers are implemented by solving local Poisson problems on domains extended into adjacent
// elements by one layer.  Thus, for an 8 x 8 x 8 brick (N = 7), one solves a 10 x 10 x 10 local problem ... using fast
// diagonalization (FDM),   u^e = (S_z x S_y x S_x) Lambda^-1 (S_z^T x S_y^T x S_x^T) b^e,   e = 1..E,   where each 1D
// matrix of eigenvectors, S_*, is 10 x 10, and Lambda is a diagonal matrix with only 1,000 nonzeros.  The leading
// complexity is ~ 12 x 10^4 operations for the application of S_* and S_*^T (implemented as dgemm), with ~ 2,000 loads
// per element (for b^e and Lambda)."  Table 2/3: `fusedFDM`, the most expensive elliptic kernel (9.5 %).
//
// Kernel (sem_fdm_dev.cuh): 12 m^4 flops on (3 m^3 + 3 m^2) values per element = 9 flop/B in FP32 at m = 10: between the
// HBM roofline and the FP32 pipe, and -- as the paper found on V100 (Table 2: limiter "S", 86 % of the L1 pipe) -- bound
// by shared-memory wavefronts when every product reads an operand from shared memory.  So the six 1-D contractions run
// in REGISTERS: a thread owns LPT whole lines of the m^3 block (m values along the contracted direction each), the rows
// of S_d are broadcast from shared memory with 128-bit loads and shared by the thread's lines, and between directions
// the block is re-distributed through shared memory once (line ownership rotates k-lines -> j-lines -> i-lines and
// back).  S_x^T, Lambda^-1 and S_x are applied by the same owner back to back, so there are 5 phases and 4 barriers.
// S, Lambda^-1 and b reach shared memory by cp.async (coalesced, no registers); u is written straight from registers.
// This is not the paper's kernel (OCCA, one thread block per element, operands in shared memory).  It is still bound
// by the shared-memory pipe (a warp-uniform 128-bit load costs two wavefronts), see DESIGN.md section 6.
#include <mutex>

#include "sem_internal.h"
#include "sem_fdm_dev.cuh"

namespace {

using namespace sem_fdm_dev;

template <typename T, int M, int LPT, int EPC, int NST, bool SREG, class IO>
int launch_cfg(sem_ctx* c, const void* S, const void* invL, const IO io) {
    using C = fdm_cfg<T, M, LPT, EPC>;
    constexpr size_t SMEM = C::SMEM1 * NST + IO::extra_bytes(EPC);
    auto kern = SREG ? k_fdm_sreg<T, M, LPT, EPC, 1, NST, IO> : k_fdm<T, M, LPT, EPC, 1, NST, IO>;
    // CTAs per SM of this instantiation, per device (the attribute is per device too); guarded for concurrent callers
    static std::mutex mu;
    static int resident_of[SEM_MAX_DEVICES] = {};
    int resident = 0;
    {
        std::lock_guard<std::mutex> lk(mu);
        const int dev = c->device >= 0 && c->device < SEM_MAX_DEVICES ? c->device : 0;
        if (!resident_of[dev] || dev != c->device) {
            if (SMEM > 48 * 1024)
                SEM_CUDA_OK(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM));
            int nb = 0;
            SEM_CUDA_OK(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, C::NT, SMEM));
            resident_of[dev] = nb > 0 ? nb : 1;
        }
        resident = resident_of[dev];
    }
    const int64_t ngrp = (c->E + C::EPC - 1) / C::EPC;
    int64_t grid = (int64_t)c->num_sms * resident;       // single wave of persistent CTAs (a grid cut down to equal
    if (grid > ngrp) grid = ngrp;                        // shares per CTA measured 8-10 % slower)
    kern<<<(unsigned)grid, C::NT, SMEM, c->stream>>>(c->E, (const T*)S, (const T*)invL, io);
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

// Configuration per (precision, m), from the variant sweeps on B200 summarised in profiles/r1e_fdm.md.
//   k_fdm:      two lines per thread wherever the registers hold them without spilling; one element per CTA at m >= 8,
//               about 128 threads' worth of elements below; one shared-memory stage (the resident CTAs hide the
//               copies) up to m = 11, two from m = 12 on (few CTAs fit).
//   k_fdm_sreg: S_d resident in registers, where it measured faster: FP32 m = 8, 10, 12 and FP64 m = 8, 10.
// FP32 tensor-core variant (k_fdm_mma): one warp per element
template <int M, class IO>
int launch_mma(sem_ctx* c, const void* S, const void* invL, const IO io) {
    using C = fdm_cfg<float, M, 1, 1>;
    const size_t smem = C::SMEM1 + IO::extra_bytes(1);
    auto kern = k_fdm_mma<M, 1, IO>;
    static std::mutex mu;
    static int resident_of[SEM_MAX_DEVICES] = {};
    int resident = 0;
    {
        std::lock_guard<std::mutex> lk(mu);
        const int dev = c->device >= 0 && c->device < SEM_MAX_DEVICES ? c->device : 0;
        if (!resident_of[dev] || dev != c->device) {
            if (smem > 48 * 1024)
                SEM_CUDA_OK(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            int nb = 0;
            SEM_CUDA_OK(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, 32, smem));
            resident_of[dev] = nb > 0 ? nb : 1;
        }
        resident = resident_of[dev];
    }
    int64_t grid = (int64_t)c->num_sms * resident;
    if (grid > c->E) grid = c->E;
    kern<<<(unsigned)grid, 32, smem, c->stream>>>(c->E, (const float*)S, (const float*)invL, io);
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

template <typename T, int M, class IO>
int launch_m(sem_ctx* c, const void* S, const void* invL, const IO io) {
    constexpr bool F32 = sizeof(T) == 4;
    if constexpr (F32 && M >= 6 && M <= 12) {
        if (c->fdm_variant == 1) return launch_mma<M, IO>(c, S, invL, io);
    }
    if constexpr (M == 8) return launch_cfg<T, M, 4, 2, 1, true, IO>(c, S, invL, io);
    else if constexpr (M == 10) return launch_cfg<T, M, 4, 1, 1, true, IO>(c, S, invL, io);
    else if constexpr (M == 12 && F32) return launch_cfg<T, M, 5, 1, 1, true, IO>(c, S, invL, io);
    else {
        constexpr int LPT = (M >= 6 && !(!F32 && M >= 12)) ? 2 : 1;
        constexpr int TPE = (M * M + LPT - 1) / LPT;
        constexpr int EPC = (M >= 8 || 128 / TPE < 1) ? 1 : 128 / TPE;
        constexpr int NST = (M >= 12 && IO::extra_bytes(1) == 0) ? 2 : 1;     // the I/O policy's area is single-staged
        return launch_cfg<T, M, LPT, EPC, NST, false, IO>(c, S, invL, io);
    }
}

template <typename T>
int launch(sem_ctx* c, int m, const void* S, const void* invL, const void* b, void* u) {
    switch (m) {
#define SEM_FDM_CASE(MM) case MM: return launch_m<T, MM>(c, S, invL, PlainIO<T, MM>{(const T*)b, (T*)u});
        SEM_FDM_CASE(2) SEM_FDM_CASE(3) SEM_FDM_CASE(4) SEM_FDM_CASE(5) SEM_FDM_CASE(6) SEM_FDM_CASE(7) SEM_FDM_CASE(8)
        SEM_FDM_CASE(9) SEM_FDM_CASE(10) SEM_FDM_CASE(11) SEM_FDM_CASE(12) SEM_FDM_CASE(13) SEM_FDM_CASE(14)
        SEM_FDM_CASE(15) SEM_FDM_CASE(16)
#undef SEM_FDM_CASE
    }
    return sem_fail(c, SEM_EINVAL, "sem_fdm_apply: m = %d outside 2..16", m);
}

// the restricted additive Schwarz smoother in one kernel: gather -> Eq. (3) -> weighted own part (SchwarzIO)
template <typename T>
int launch_schwarz(sem_ctx* c, int m, const void* S, const void* invL, const void* r, const int4* link,
                   const int32_t* nrm, const void* W, void* z) {
    switch (m) {
#define SEM_FDM_CASE(MM) \
    case MM: return launch_m<T, MM>(c, S, invL, SchwarzIO<T, MM>{(const T*)r, link, nrm, (const T*)W, (T*)z});
        SEM_FDM_CASE(4) SEM_FDM_CASE(5) SEM_FDM_CASE(6) SEM_FDM_CASE(7) SEM_FDM_CASE(8) SEM_FDM_CASE(9) SEM_FDM_CASE(10)
        SEM_FDM_CASE(11) SEM_FDM_CASE(12) SEM_FDM_CASE(13) SEM_FDM_CASE(14) SEM_FDM_CASE(15) SEM_FDM_CASE(16)
#undef SEM_FDM_CASE
    }
    return sem_fail(c, SEM_EINVAL, "Schwarz local solve: m = %d outside 4..16", m);
}

}  // namespace

extern "C" int sem_fdm_apply(sem_ctx* ctx, int m, const void* S, const void* inv_lambda, const void* b, void* u,
                             sem_prec prec) {
    if (!ctx) return SEM_EINVAL;
    ctx->err.clear();
    if (!S || !inv_lambda || !b || !u) return sem_fail(ctx, SEM_EINVAL, "sem_fdm_apply: NULL pointer");
    if (prec != SEM_F64 && prec != SEM_F32) return sem_fail(ctx, SEM_EINVAL, "sem_fdm_apply: bad sem_prec");
    if (m < 2 || m > 16) return sem_fail(ctx, SEM_EINVAL, "sem_fdm_apply: m = %d outside 2..16", m);
    if ((((uintptr_t)S | (uintptr_t)inv_lambda | (uintptr_t)b | (uintptr_t)u) & 15) != 0)
        return sem_fail(ctx, SEM_EINVAL, "sem_fdm_apply: S, inv_lambda, b, u must be 16-byte aligned");
    if (prec == SEM_F64) return launch<double>(ctx, m, S, inv_lambda, b, u);
    return launch<float>(ctx, m, S, inv_lambda, b, u);
}

// NEXT-2b, restricted variant fused (sem_schwarz.cu): z_L = W (A~^-1 R r)|own nodes, straight from r, no block in HBM
int sem_launch_fdm_schwarz(sem_ctx* c, int m, const void* S, const void* invL, const void* r, const int4* link,
                           const int32_t* nrm, const void* W, void* z, sem_prec prec) {
    if (prec == SEM_F64) return launch_schwarz<double>(c, m, S, invL, r, link, nrm, W, z);
    return launch_schwarz<float>(c, m, S, invL, r, link, nrm, W, z);
}
