// sem_transfer.cu — NEXT-1: p-multigrid transfer operators between two discretisations (orders
// N_c <= N_f) of the same E elements.  P:103: "Coarse-to-fine interpolations are cast as efficient tensor contractions,
// u_f = (J x J x J) u_c, where J is the 1D polynomial interpolation operator from the coarse GLL points to the fine GLL
// points ... only a single J matrix (of size N+1 or less) is needed for the entire domain, for each pMG level."
// Restriction is the transpose, r_c = (J^T x J^T x J^T) r_f.  Element by element, local layout, no gather-scatter.
//
// Sum-factorised: three 1-D contractions through shared memory (i, then j, then k), J in shared memory.  The work is
// tiny and the kernel is bound by the read of p_in^3 and the write of p_out^3 values per element (and, at the paper's
// E ~ 7000 per GPU, by launch latency), so the orders are run-time values: one kernel for every level pair.
#include "sem_internal.h"

namespace {

constexpr int TNT = 128;

// For each of `ne` elements (element strides es_dst / es_src):  dst[o2][o1][o0] = sum over the contracted axis of
// M * src[n2][n1][n0];  AXIS 0/1/2 = i/j/k (i fastest).  TRANSPOSED = false: M = J used as J[out][in] (prolongation);
// true: J[in][out] (restriction).  J is [pf][pc].
template <typename T, int AXIS, bool TRANSPOSED>
__device__ __forceinline__ void contract(T* __restrict__ dst, int64_t es_dst, const T* __restrict__ src, int es_src,
                                         const T* __restrict__ J, int pc, int ne, int n0, int n1, int n2, int nin,
                                         int nout, bool accumulate = false) {
    const int o0 = AXIS == 0 ? nout : n0, o1 = AXIS == 1 ? nout : n1, o2 = AXIS == 2 ? nout : n2;
    const int per = o0 * o1 * o2, total = per * ne;
    const int sstride = AXIS == 0 ? 1 : AXIS == 1 ? n0 : n0 * n1;
    for (int t = threadIdx.x; t < total; t += TNT) {
        const int el = t / per, q = t - el * per;
        const int a0 = q % o0, a1 = (q / o0) % o1, a2 = q / (o0 * o1);
        const int out = AXIS == 0 ? a0 : AXIS == 1 ? a1 : a2;
        const T* sp = src + el * es_src + (AXIS == 0 ? 0 : a0) + n0 * ((AXIS == 1 ? 0 : a1) + n1 * (AXIS == 2 ? 0 : a2));
        const T* jp = TRANSPOSED ? J + out : J + out * pc;
        const int jstride = TRANSPOSED ? pc : 1;
        T s = accumulate ? dst[el * es_dst + q] : T(0);      // loaded before the contraction, which hides its latency
        for (int l = 0; l < nin; ++l) s += jp[l * jstride] * sp[l * sstride];
        dst[el * es_dst + q] = s;
    }
}

// One CTA works on `epc` consecutive elements at a time so that small orders still fill its threads.
// PC, PF > 0: the level pair is known at compile time (index arithmetic folds, loops unroll); 0: run-time orders.
template <typename T, bool RESTRICT, int PC, int PF>
__global__ void __launch_bounds__(TNT) k_transfer(int64_t E, int pc_rt, int pf_rt, int epc_rt, const T* __restrict__ Jg,
                                                  const T* __restrict__ in, T* __restrict__ out,
                                                  const T* __restrict__ in_minus, const double* __restrict__ wt) {
    // Fused forms used by the V-cycle (sem_pmg.cu), wt = 1/multiplicity, 0 at Dirichlet nodes (fine level):
    //   RESTRICT with in_minus:  input = (in - in_minus) * wt         (weighted residual, never materialised)
    //   PROLONG  with wt:        out  += result                        (coarse correction added in place; a
    //                            correction that vanishes at the coarse Dirichlet nodes prolongs to exact zeros at the
    //                            fine ones -- J has exact 0 / 1 entries at the end points -- so no mask is needed)
    const int pc = PC > 0 ? PC : pc_rt, pf = PF > 0 ? PF : pf_rt;
    const int epc = PF > 0 ? (TNT / (PF * PF) > 0 ? TNT / (PF * PF) : 1) : epc_rt;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sJ = reinterpret_cast<T*>(smem_raw);
    const int pin = RESTRICT ? pf : pc, pout = RESTRICT ? pc : pf;
    const int big = pf * pf * pf;
    T* bufA = sJ + ((pf * pc + 3) & ~3);
    T* bufB = bufA + epc * big;
    for (int t = threadIdx.x; t < pf * pc; t += TNT) sJ[t] = Jg[t];
    const int nin3 = pin * pin * pin;
    const int64_t nout3 = (int64_t)pout * pout * pout;
    const int64_t ngrp = (E + epc - 1) / epc;
    for (int64_t g = blockIdx.x; g < ngrp; g += gridDim.x) {
        const int64_t e0 = g * epc;
        const int ne = (int)(E - e0 < epc ? E - e0 : epc);
        __syncthreads();                                   // bufA free (and sJ filled, first time round)
        if (RESTRICT && in_minus) {
            for (int t = threadIdx.x; t < ne * nin3; t += TNT)
                bufA[t] = (in[e0 * nin3 + t] - in_minus[e0 * nin3 + t]) * (T)wt[e0 * nin3 + t];
        } else {
            for (int t = threadIdx.x; t < ne * nin3; t += TNT) bufA[t] = in[e0 * nin3 + t];     // contiguous elements
        }
        __syncthreads();
        contract<T, 0, RESTRICT>(bufB, big, bufA, nin3, sJ, pc, ne, pin, pin, pin, pin, pout);      // [pin][pin][pout]
        __syncthreads();
        contract<T, 1, RESTRICT>(bufA, big, bufB, big, sJ, pc, ne, pout, pin, pin, pin, pout);      // [pin][pout][pout]
        __syncthreads();
        contract<T, 2, RESTRICT>(out + e0 * nout3, nout3, bufA, big, sJ, pc, ne, pout, pout, pin, pin, pout,
                                 !RESTRICT && wt != nullptr);
    }
}

// J[i][j] = coarse Lagrange cardinal function j at fine point i, by the barycentric formula (host, long double)
void interp_matrix(const sem_ctx* cc, const sem_ctx* cf, double* J) {
    const int pc = cc->p, pf = cf->p;
    long double wb[SEM_MAXP];
    for (int j = 0; j < pc; ++j) {
        long double d = 1.0L;
        for (int m = 0; m < pc; ++m) if (m != j) d *= (long double)cc->xi[j] - (long double)cc->xi[m];
        wb[j] = 1.0L / d;
    }
    for (int i = 0; i < pf; ++i) {
        const long double x = cf->xi[i];
        int hit = -1;
        for (int j = 0; j < pc; ++j) if (x == (long double)cc->xi[j]) hit = j;
        if (hit >= 0) {
            for (int j = 0; j < pc; ++j) J[i * pc + j] = j == hit ? 1.0 : 0.0;
            continue;
        }
        long double den = 0.0L;
        for (int j = 0; j < pc; ++j) den += wb[j] / (x - (long double)cc->xi[j]);
        for (int j = 0; j < pc; ++j) J[i * pc + j] = (double)((wb[j] / (x - (long double)cc->xi[j])) / den);
    }
}

constexpr size_t J_SLOT_BYTES = sizeof(double) * SEM_MAXP * SEM_MAXP;

template <typename T>
int launch(sem_ctx* cf, int pc, const double* Jh, const void* in, void* out, bool restrict_, const void* in_minus,
           const double* wt) {
    const int pf = cf->p;
    // One device copy of J per (coarse p, precision), each in its own slot of d_J and written once: a CUDA graph that
    // recorded a transfer keeps pointing at a matrix that no later call with another level pair or precision rewrites.
    const int key = pc * 2 + (sizeof(T) == 8 ? 0 : 1);
    const T* dJ = reinterpret_cast<const T*>(static_cast<const char*>(cf->d_J) + (size_t)key * J_SLOT_BYTES);
    if (!((cf->J_have >> key) & 1ull)) {
        T hJ[SEM_MAXP * SEM_MAXP];
        for (int q = 0; q < pf * pc; ++q) hJ[q] = (T)Jh[q];          // S16: computed in double, rounded once
        SEM_CUDA_OK(cf, cudaMemcpy(const_cast<T*>(dJ), hJ, sizeof(T) * pf * pc, cudaMemcpyHostToDevice));
        cf->J_have |= 1ull << key;
    }
    int epc = TNT / (pf * pf);
    if (epc < 1) epc = 1;
    const size_t smem = sizeof(T) * (((size_t)(pf * pc + 3) & ~(size_t)3) + 2 * (size_t)epc * pf * pf * pf);
    // the level pairs of config 4 (N = 7-3-1) and of the paper's schedules 8-5-1 and 8-6-4-1 are specialised
    using kern_t = void (*)(int64_t, int, int, int, const T*, const T*, T*, const T*, const double*);
    kern_t kern = restrict_ ? k_transfer<T, true, 0, 0> : k_transfer<T, false, 0, 0>;
#define SEM_TR_CASE(A, B) \
    if (pc == A && pf == B) kern = restrict_ ? k_transfer<T, true, A, B> : k_transfer<T, false, A, B>;
    SEM_TR_CASE(2, 4) SEM_TR_CASE(4, 8) SEM_TR_CASE(2, 8) SEM_TR_CASE(2, 6) SEM_TR_CASE(6, 9) SEM_TR_CASE(2, 5)
    SEM_TR_CASE(5, 7) SEM_TR_CASE(7, 9)
#undef SEM_TR_CASE
    if (smem > 48 * 1024) SEM_CUDA_OK(cf, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int64_t ngrp = (cf->E + epc - 1) / epc;
    int64_t grid = (int64_t)cf->num_sms * 8;
    if (grid > ngrp) grid = ngrp;
    kern<<<(unsigned)grid, TNT, smem, cf->stream>>>(cf->E, pc, pf, epc, dJ, (const T*)in, (T*)out,
                                                    (const T*)in_minus, wt);
    SEM_CUDA_OK(cf, cudaGetLastError());
    return SEM_OK;
}

int check_pair(sem_ctx* cc, sem_ctx* cf) {
    if (!cc || !cf) return SEM_EINVAL;
    cf->err.clear();
    if (cc->E != cf->E) return sem_fail(cf, SEM_EINVAL, "sem_transfer: contexts have different element counts");
    if (cc->N > cf->N) return sem_fail(cf, SEM_EINVAL, "sem_transfer: coarse order exceeds fine order");
    return SEM_OK;
}

}  // namespace

extern "C" int sem_get_interp(sem_ctx* coarse, sem_ctx* fine, double* J) {
    int rc = check_pair(coarse, fine);
    if (rc) return rc;
    if (!J) return sem_fail(fine, SEM_EINVAL, "sem_get_interp: NULL buffer");
    interp_matrix(coarse, fine, J);
    return SEM_OK;
}

// in_minus / wt: the fused forms documented at k_transfer (internal callers only; the public call passes none)
int sem_launch_transfer(sem_ctx* coarse, sem_ctx* fine, const void* in, void* out, sem_prec prec, sem_transfer_dir dir,
                        const void* in_minus, const double* wt) {
    int rc = check_pair(coarse, fine);
    if (rc) return rc;
    if (!in || !out || in == out) return sem_fail(fine, SEM_EINVAL, "sem_transfer: NULL or aliased vectors");
    if (prec != SEM_F64 && prec != SEM_F32) return sem_fail(fine, SEM_EINVAL, "sem_transfer: bad sem_prec");
    if (dir != SEM_PROLONG && dir != SEM_RESTRICT) return sem_fail(fine, SEM_EINVAL, "sem_transfer: bad direction");
    if (!fine->d_J) SEM_CUDA_OK(fine, cudaMalloc((void**)&fine->d_J, J_SLOT_BYTES * (2 * SEM_MAXP + 2)));
    double Jh[SEM_MAXP * SEM_MAXP];
    interp_matrix(coarse, fine, Jh);
    if (prec == SEM_F64) return launch<double>(fine, coarse->p, Jh, in, out, dir == SEM_RESTRICT, in_minus, wt);
    return launch<float>(fine, coarse->p, Jh, in, out, dir == SEM_RESTRICT, in_minus, wt);
}

extern "C" int sem_transfer(sem_ctx* coarse, sem_ctx* fine, const void* in, void* out, sem_prec prec,
                            sem_transfer_dir dir) {
    return sem_launch_transfer(coarse, fine, in, out, prec, dir, nullptr, nullptr);
}
