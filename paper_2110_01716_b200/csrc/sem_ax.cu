// sem_ax.cu — a3-a5 (+a9): the local spectral-element operator  w = D^T G D u (+ lambda B u), element by element.
// P:93 (footnote): u_r,ijk = sum_l D_il u_ljk, "an Np x Np matrix times an Np x Np^2 matrix"; O4 for the
// full operator; S16 for FP32.  12p+15 flops and 64 B (FP64) / 32 B (FP32) of compulsory HBM traffic per node: the
// kernel is HBM-bound, so the design is about keeping enough bytes in flight and keeping shared-memory and FP64-issue
// pressure below the HBM rate:
//   * thread (i,j) owns the k-column of one element: u[.][j][i] and the w accumulators live in registers, so the t
//     direction never touches shared memory and D[k][l] for it is a compile-time constant-bank operand;
//   * the rows D[i][.], D[j][.], D[.][i], D[.][j] the thread needs for r and s stay in registers for the whole kernel;
//   * G is stored slab-major (sem_geom.cu) and streamed through a ring of shared-memory stages by bulk async copies
//     (cp.async.bulk + mbarrier transaction counts, evict-first in L2) issued NS slabs ahead, so the bytes in flight per
//     SM do not depend on registers or occupancy;  u arrives the same way, double-buffered per element;
//   * persistent CTAs (one element group at a time, grid = SMs x resident CTAs) write w straight from registers.
// That is ax_stream (every p <= 12; odd p takes u by plain loads).  At p = 8 -- the paper's N = 7 -- the r and s
// contractions run on the tensor cores instead, one WARP per element with the same streaming ring: ax_dmma (FP64,
// mma.sync m8n8k4; the measured DMMA path north_star asks for: it won), ax_tf32 (FP32, m16n8k8 TF32 in three passes),
// ax_dmma_many (2 or 3 fields sharing one pass over G).  Kernels in this file, in order: ax_simple, ax_stream, ax_pencil
// (a measured alternative for p >= 8, one pencil of p values per thread and contraction), ax_dmma, ax_tf32,
// ax_dmma_many; then the launchers and the chunked operator / gather-scatter driver (sem_launch_ax_gs).
// ax_simple is the plain-load version of the same arithmetic: p > 12 and unaligned pointers use it.  a9 (G recomputed
// from the 8 trilinear vertices inside the kernel): ax_dmma_rg for FP64 p = 8, ax_stream<..., RG> for p <= 12, ax_simple beyond.
#include <array>
#include <map>
#include <mutex>
#include <type_traits>

#include "sem_geom_dev.cuh"
#include "sem_internal.h"

namespace {

// ---------------------------------------------------------------------------------------------------------------
// PTX helpers (sm_90+/sm_100a): mbarrier + bulk async copy global -> shared
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar,
                                         uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::
            "r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}

// ---------------------------------------------------------------------------------------------------------------
// shared pieces
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int P>
struct DParam {            // by-value kernel parameter: constant bank
    T D[P * P];            // D[i*P + l] = dh_l/dr(xi_i)
};

template <int P> constexpr int epb_of() { return P * P >= 64 ? 1 : (64 + P * P - 1) / (P * P); }
template <int P> constexpr int threads_of() { return ((epb_of<P>() * P * P + 31) / 32) * 32; }

// read P consecutive values starting at a pointer whose byte offset is a multiple of P*sizeof(T)
template <typename T, int P>
__device__ __forceinline__ void load_row(const T* __restrict__ ptr, T (&out)[P]) {
    if constexpr ((P * sizeof(T)) % 16 == 0) {
        constexpr int V = 16 / sizeof(T);
        using VT = typename std::conditional<sizeof(T) == 8, double2, float4>::type;
#pragma unroll
        for (int v = 0; v < P / V; ++v) {
            const VT q = reinterpret_cast<const VT*>(ptr)[v];
            if constexpr (sizeof(T) == 8) { out[2 * v] = q.x; out[2 * v + 1] = q.y; }
            else { out[4 * v] = q.x; out[4 * v + 1] = q.y; out[4 * v + 2] = q.z; out[4 * v + 3] = q.w; }
        }
    } else if constexpr (sizeof(T) == 4 && (P * sizeof(T)) % 8 == 0) {
#pragma unroll
        for (int v = 0; v < P / 2; ++v) {
            const float2 q = reinterpret_cast<const float2*>(ptr)[v];
            out[2 * v] = q.x; out[2 * v + 1] = q.y;
        }
    } else {
#pragma unroll
        for (int l = 0; l < P; ++l) out[l] = ptr[l];
    }
}

// The four 1-D rows/columns of D a thread (i,j) keeps in registers.
template <typename T, int P>
struct DRows {
    T Di[P], Dj[P], DTi[P], DTj[P];
    __device__ __forceinline__ void init(const DParam<T, P>& dp, int i, int j) {
#pragma unroll
        for (int l = 0; l < P; ++l) {
            Di[l] = dp.D[i * P + l];
            Dj[l] = dp.D[j * P + l];
            DTi[l] = dp.D[l * P + i];
            DTj[l] = dp.D[l * P + j];
        }
        // pin the rows in registers: without this the compiler re-reads them with indexed constant loads (LDC
        // c[0x0][R+..]) inside the slab loop, and the indexed-constant cache becomes the busiest unit of the SM
#pragma unroll
        for (int l = 0; l < P; ++l) {
            if constexpr (sizeof(T) == 8)
                asm volatile("" : "+d"(Di[l]), "+d"(Dj[l]), "+d"(DTi[l]), "+d"(DTj[l]));
            else
                asm volatile("" : "+f"(Di[l]), "+f"(Dj[l]), "+f"(DTi[l]), "+f"(DTj[l]));
        }
    }
    // Same rows from a shared-memory copy sD[P*P] of D, read with volatile loads: values that come out of a volatile
    // asm cannot be re-materialised from the constant bank, so ptxas has to keep them in registers whatever else the
    // kernel contains (with init() that holds only as long as nothing else in the kernel raises register pressure).
    __device__ __forceinline__ void init_shared(const T* sD, int i, int j) {
        const uint32_t base = (uint32_t)__cvta_generic_to_shared(sD);
#pragma unroll
        for (int l = 0; l < P; ++l) {
            Di[l] = lds_volatile(base + (uint32_t)((i * P + l) * sizeof(T)));
            Dj[l] = lds_volatile(base + (uint32_t)((j * P + l) * sizeof(T)));
            DTi[l] = lds_volatile(base + (uint32_t)((l * P + i) * sizeof(T)));
            DTj[l] = lds_volatile(base + (uint32_t)((l * P + j) * sizeof(T)));
        }
    }
    static __device__ __forceinline__ T lds_volatile(uint32_t addr) {
        T v;
        if constexpr (sizeof(T) == 8) asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
        else asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
        return v;
    }
};

// One k-slab of the operator for thread (i,j) of one element.
//   su: the element's u in shared memory [P][P][P];  uk/wk: the thread's k-column of u / accumulators of w.
//   g[6]: this node's factors.  sgr/sgs: this element's exchange buffers for slab parity `buf` ([P*P] each).
// The caller synchronises the element's threads between part1 and part2.
template <typename T, int P>
__device__ __forceinline__ void slab_part1(const DParam<T, P>& dp, const DRows<T, P>& dr, const T* __restrict__ su,
                                           const T (&uk)[P], T (&wk)[P], const T (&g)[6], int k, int i, int j,
                                           T& gr_out, T& gs_out) {
    T row[P];
    load_row<T, P>(su + (k * P + j) * P, row);
    const T* col = su + k * P * P + i;
    T ur = T(0), us = T(0), ut = T(0);
#pragma unroll
    for (int l = 0; l < P; ++l) {
        ur += dr.Di[l] * row[l];                 // u_r = sum_l D[i][l] u[k][j][l]
        us += dr.Dj[l] * col[l * P];             // u_s = sum_l D[j][l] u[k][l][i]
        ut += dp.D[k * P + l] * uk[l];           // u_t = sum_l D[k][l] u[l][j][i]
    }
    gr_out = g[0] * ur + g[1] * us + g[2] * ut;
    gs_out = g[1] * ur + g[3] * us + g[4] * ut;
    const T gt = g[2] * ur + g[4] * us + g[5] * ut;
#pragma unroll
    for (int l = 0; l < P; ++l) wk[l] += dp.D[k * P + l] * gt;   // w[l][j][i] += D[k][l] g_t[k][j][i]
}

template <typename T, int P>
__device__ __forceinline__ T slab_part2(const DRows<T, P>& dr, int i, int j, const T* __restrict__ sgr,
                                        const T* __restrict__ sgs) {
    T row[P];
    load_row<T, P>(sgr + j * P, row);
    T ar = T(0), as = T(0);                      // two independent chains
#pragma unroll
    for (int l = 0; l < P; ++l) {
        ar += dr.DTi[l] * row[l];                // sum_l D[l][i] g_r[k][j][l]
        as += dr.DTj[l] * sgs[l * P + i];        // sum_l D[l][j] g_s[k][l][i]
    }
    return ar + as;
}

// ---- a9 inside the streaming kernel: the geometric factors of a node recomputed from the element's 8 vertices ----
template <typename T, int P>
struct GllP { T xi[P], rho[P]; };            // by value: compile-time indices come from the constant bank

// Column (i, j) of a trilinear element (S5): x_r = Ja + Jb t, x_s = Jc + Jd t, x_t = Je for all nodes of the column
template <typename T>
struct ColJac { T Ja[3], Jb[3], Jc[3], Jd[3], Je[3], Wij; };

template <typename T>
__device__ __forceinline__ void col_jac_init(const double* __restrict__ vert_e, bool active, T r, T s, T Wij,
                                             ColJac<T>& cj) {
    double X[8][3], cf[8][3];
#pragma unroll
    for (int v = 0; v < 8; ++v)
#pragma unroll
        for (int d = 0; d < 3; ++d) X[v][d] = active ? __ldg(vert_e + v * 3 + d) : (double)((v >> d) & 1);
    sem_trilinear_coef(X, cf);               // vertex differences in FP64 even on the FP32 path (no cancellation)
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        cj.Ja[d] = (T)cf[1][d] + (T)cf[4][d] * s;
        cj.Jb[d] = (T)cf[5][d] + (T)cf[7][d] * s;
        cj.Jc[d] = (T)cf[2][d] + (T)cf[4][d] * r;
        cj.Jd[d] = (T)cf[6][d] + (T)cf[7][d] * r;
        cj.Je[d] = (T)cf[3][d] + (T)cf[5][d] * r + ((T)cf[6][d] + (T)cf[7][d] * r) * s;
    }
    cj.Wij = Wij;
}

// (g_r, g_s, g_t) = G (u_r, u_s, u_t) at t = tk, W = Wij rho_k, without forming G:  G = (W / det) A A^T with the adjugate
// rows a_0 = x_s x x_t, a_1 = x_t x x_r, a_2 = x_r x x_s, so G v = (W / det) A (A^T v); det = x_r . a_0
template <typename T>
__device__ __forceinline__ void col_jac_apply(const ColJac<T>& cj, T tk, T rk, T ur, T us, T ut, T& gr, T& gs, T& gt) {
    T xr[3], xs[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) { xr[d] = cj.Ja[d] + cj.Jb[d] * tk; xs[d] = cj.Jc[d] + cj.Jd[d] * tk; }
    const T* xt = cj.Je;
    const T a0x = xs[1] * xt[2] - xs[2] * xt[1], a0y = xs[2] * xt[0] - xs[0] * xt[2], a0z = xs[0] * xt[1] - xs[1] * xt[0];
    const T a1x = xt[1] * xr[2] - xt[2] * xr[1], a1y = xt[2] * xr[0] - xt[0] * xr[2], a1z = xt[0] * xr[1] - xt[1] * xr[0];
    const T a2x = xr[1] * xs[2] - xr[2] * xs[1], a2y = xr[2] * xs[0] - xr[0] * xs[2], a2z = xr[0] * xs[1] - xr[1] * xs[0];
    const T det = xr[0] * a0x + xr[1] * a0y + xr[2] * a0z;
    T rdet;
    if constexpr (sizeof(T) == 8) rdet = __drcp_rn(det); else rdet = __frcp_rn(det);
    const T sc = cj.Wij * rk * rdet;
    const T zx = a0x * ur + a1x * us + a2x * ut;
    const T zy = a0y * ur + a1y * us + a2y * ut;
    const T zz = a0z * ur + a1z * us + a2z * ut;
    gr = sc * (a0x * zx + a0y * zy + a0z * zz);
    gs = sc * (a1x * zx + a1y * zy + a1z * zz);
    gt = sc * (a2x * zx + a2y * zy + a2z * zz);
}

// slab_part1 with the factors recomputed (same contractions)
template <typename T, int P>
__device__ __forceinline__ void slab_part1_rg(const DParam<T, P>& dp, const DRows<T, P>& dr, const T* __restrict__ su,
                                              const T (&uk)[P], T (&wk)[P], const ColJac<T>& cj, T tk, T rk, int k, int i,
                                              int j, T& gr_out, T& gs_out) {
    T row[P];
    load_row<T, P>(su + (k * P + j) * P, row);
    const T* col = su + k * P * P + i;
    T ur = T(0), us = T(0), ut = T(0);
#pragma unroll
    for (int l = 0; l < P; ++l) {
        ur += dr.Di[l] * row[l];
        us += dr.Dj[l] * col[l * P];
        ut += dp.D[k * P + l] * uk[l];
    }
    T gt;
    col_jac_apply<T>(cj, tk, rk, ur, us, ut, gr_out, gs_out, gt);
#pragma unroll
    for (int l = 0; l < P; ++l) wk[l] += dp.D[k * P + l] * gt;
}

template <typename T>
__device__ __forceinline__ void block_dot_flush(T partial, double* __restrict__ dot_out) {
    __shared__ double red[32];
    double v = (double)partial;
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) red[warp] = v;
    __syncthreads();
    if (warp == 0) {
        v = lane < nw ? red[lane] : 0.0;
        for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) atomicAdd(dot_out, v);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// ax_simple: plain loads.  RECOMP: G from the trilinear vertices (a9).
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int P, bool RECOMP>
__global__ void __launch_bounds__(threads_of<P>()) ax_simple(int64_t E, DParam<T, P> dp, Gll1D gll, int64_t slab,
                                                             const T* __restrict__ Gs, const double* __restrict__ vert,
                                                             const T* __restrict__ Bm, T lambda,
                                                             const T* __restrict__ u, T* __restrict__ w,
                                                             const int* __restrict__ skip_flag,
                                                             double* __restrict__ dot_out) {
    constexpr int EPB = epb_of<P>(), P2 = P * P, P3 = P2 * P;
    __shared__ __align__(16) T su[EPB * P3];
    __shared__ __align__(16) T sgr[2][EPB * P2];
    __shared__ __align__(16) T sgs[2][EPB * P2];
    if (skip_flag && *skip_flag) return;
    const int tid = threadIdx.x;
    const bool lane_ok = tid < EPB * P2;
    const int slot = lane_ok ? tid / P2 : 0;
    const int ij = lane_ok ? tid % P2 : 0;
    const int j = ij / P, i = ij % P;
    DRows<T, P> dr;
    dr.init(dp, i, j);
    T partial = T(0);
    const int64_t ngroups = (E + EPB - 1) / EPB;
    for (int64_t grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
        const int64_t e = grp * EPB + slot;
        const bool active = lane_ok && e < E;
        T uk[P], wk[P];
#pragma unroll
        for (int k = 0; k < P; ++k) {
            uk[k] = active ? u[e * P3 + k * P2 + ij] : T(0);
            wk[k] = T(0);
            if (lane_ok) su[slot * P3 + k * P2 + ij] = uk[k];
        }
        // recomputed G: per-thread pieces of the trilinear Jacobian that do not depend on k (r = xi_i, s = xi_j)
        T Ja[3], Jb[3], Jc[3], Jd[3], Je[3];
        if constexpr (RECOMP) {
            double X[8][3], cf[8][3];
#pragma unroll
            for (int v = 0; v < 8; ++v)
#pragma unroll
                for (int d = 0; d < 3; ++d) X[v][d] = active ? vert[(e * 8 + v) * 3 + d] : (double)((v >> d) & 1);
            sem_trilinear_coef(X, cf);       // vertex differences in FP64 even on the FP32 path (no cancellation)
            const T r = (T)gll.xi[i], s = (T)gll.xi[j];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                Ja[d] = (T)cf[1][d] + (T)cf[4][d] * s;          // dx/dr = Ja + Jb t
                Jb[d] = (T)cf[5][d] + (T)cf[7][d] * s;
                Jc[d] = (T)cf[2][d] + (T)cf[4][d] * r;          // dx/ds = Jc + Jd t
                Jd[d] = (T)cf[6][d] + (T)cf[7][d] * r;
                Je[d] = (T)cf[3][d] + (T)cf[5][d] * r + ((T)cf[6][d] + (T)cf[7][d] * r) * s;   // dx/dt
            }
        }
        __syncthreads();
        const T* sue = su + slot * P3;
#pragma unroll
        for (int k = 0; k < P; ++k) {
            T g[6];
            if constexpr (RECOMP) {
                const T t = (T)gll.xi[k];
                T J[3][3], B;
#pragma unroll
                for (int d = 0; d < 3; ++d) { J[d][0] = Ja[d] + Jb[d] * t; J[d][1] = Jc[d] + Jd[d] * t; J[d][2] = Je[d]; }
                sem_factors<T>(J, (T)(gll.rho[i] * gll.rho[j] * gll.rho[k]), g, B);
            } else {
#pragma unroll
                for (int c = 0; c < 6; ++c) g[c] = active ? Gs[sem_g_off(e, k, P, EPB, slab) + c * P2 + ij] : T(0);
            }
            const int buf = k & 1;
            if (lane_ok) {
                T gr, gs;
                slab_part1<T, P>(dp, dr, sue, uk, wk, g, k, i, j, gr, gs);
                sgr[buf][slot * P2 + ij] = gr;
                sgs[buf][slot * P2 + ij] = gs;
            }
            __syncthreads();
            if (lane_ok) wk[k] += slab_part2<T, P>(dr, i, j, sgr[buf] + slot * P2, sgs[buf] + slot * P2);
        }
        if (active) {
#pragma unroll
            for (int k = 0; k < P; ++k) {
                T v = wk[k];
                if (Bm) v += lambda * Bm[e * P3 + k * P2 + ij] * uk[k];
                w[e * P3 + k * P2 + ij] = v;
                partial += uk[k] * v;
            }
        }
        __syncthreads();     // su is rewritten by the next group
    }
    if (dot_out) block_dot_flush(partial, dot_out);
}

// ---------------------------------------------------------------------------------------------------------------
// ax_stream: persistent CTAs, G slabs and u elements arrive by bulk async copies into shared-memory rings.
// Any P <= 12 and 16-byte aligned u.  The G slabs are padded to 16 bytes (sem_geom.cu) and always arrive by bulk copies;
// u arrives by bulk copies when an element block is a multiple of 16 bytes (even p), by plain loads otherwise (odd p).
//
template <typename T, int P, int NS, bool RG = false>
struct StreamSmem {
    static constexpr int EPB = epb_of<P>(), P2 = P * P, P3 = P2 * P;
    // values per element slab, padded to 16 bytes (sem_geom.cu: slab_f64 / slab_f32): only FP32 with odd p needs the pad
    static constexpr int SLAB = 6 * P2 + ((6 * P2 * (int)sizeof(T)) % 16 ? 2 : 0);
    static constexpr bool UBULK = (P3 * (int)sizeof(T)) % 16 == 0;   // element blocks of u are 16-byte multiples: bulk copies
    alignas(128) T g[RG ? 1 : NS][RG ? 16 : EPB * SLAB];     // RG (recomputed factors, a9): no G ring
    alignas(128) T u[2][EPB * P3];
    alignas(16) T sgr[2][EPB * P2];
    alignas(16) T sgs[2][EPB * P2];
    alignas(8) uint64_t gfull[NS];
    alignas(8) uint64_t ufull[2];
    alignas(16) T D[P * P];                                  // copy of D for DRows::init_shared
    alignas(16) T xr[2 * P];                                 // RG: xi, rho for the thread-dependent indices i, j
};

// RG = true (a9): the factors are recomputed per node from the element's vertices (col_jac_*), Gs is not read, `vert`
// points at the first element's 8 vertices and gl holds the GLL points / weights.
template <typename T, int P, int NS, int MINB, bool RG = false>
__global__ void __launch_bounds__(threads_of<P>(), MINB) ax_stream(int64_t E, DParam<T, P> dp,
                                                                   const T* __restrict__ Gs, const T* __restrict__ Bm,
                                                                   T lambda, const T* __restrict__ u,
                                                                   T* __restrict__ w, const int* __restrict__ skip_flag,
                                                                   double* __restrict__ dot_out, int u_keep,
                                                                   const double* __restrict__ vert, GllP<T, P> gl) {
    using SM = StreamSmem<T, P, NS, RG>;
    constexpr int EPB = SM::EPB, P2 = SM::P2, P3 = SM::P3, SLAB = SM::SLAB, NT = threads_of<P>();
    constexpr bool FULL = EPB * P2 == NT;           // every thread owns a column
    constexpr uint32_t GBYTES = EPB * SLAB * sizeof(T);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    SM& sm = *reinterpret_cast<SM*>(smem_raw);
    if (skip_flag && *skip_flag) return;
    const int tid = threadIdx.x;
    const bool lane_ok = FULL || tid < EPB * P2;
    const int slot = lane_ok ? tid / P2 : 0;
    const int ij = lane_ok ? tid % P2 : 0;
    const int j = ij / P, i = ij % P;

    constexpr bool UBULK = SM::UBULK;               // odd p: u arrives by plain loads (its blocks are not 16-byte multiples)
    const int64_t ngroups = (E + EPB - 1) / EPB;
    const int64_t nmine = blockIdx.x < ngroups ? (ngroups - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const int tail_n = (int)(E - (ngroups - 1) * EPB);          // elements of the globally last group

    // ---- producer (thread 0): slabs are issued in consumption order, NS ahead; G is padded to whole groups ----
    const T* gsrc = Gs + (int64_t)blockIdx.x * (P * EPB * SLAB);
    const int64_t gjump = (int64_t)(gridDim.x - 1) * (P * EPB * SLAB);
    int64_t gleft = RG ? 0 : nmine * P;
    uint64_t pol_g = 0, pol_u = 0;
    auto issue_u = [&](int64_t n) {
        const int64_t grp = blockIdx.x + n * gridDim.x;
        const uint32_t bytes = (uint32_t)((grp == ngroups - 1 ? tail_n : EPB) * P3 * sizeof(T));
        const int b = (int)(n & 1);
        mbar_expect_tx(&sm.ufull[b], bytes);
        bulk_g2s(&sm.u[b][0], u + grp * (EPB * P3), bytes, &sm.ufull[b], pol_u);
    };
    if (tid == 0) {
#pragma unroll
        for (int q = 0; q < NS; ++q) mbar_init(&sm.gfull[q], 1);
        mbar_init(&sm.ufull[0], 1);
        mbar_init(&sm.ufull[1], 1);
        mbar_fence_init();
    }
    for (int t = tid; t < P * P; t += NT) sm.D[t] = dp.D[t];
    if constexpr (RG) {
#pragma unroll
        for (int q = 0; q < P; ++q)
            if (tid == q) { sm.xr[q] = gl.xi[q]; sm.xr[P + q] = gl.rho[q]; }
    }
    __syncthreads();
    if (tid == 0 && nmine > 0) {
        pol_g = policy_evict_first();
        pol_u = u_keep ? policy_evict_last() : policy_evict_first();
        if (UBULK) issue_u(0);
        int gk = 0;
        for (int q = 0; q < NS && gleft > 0; ++q) {
            mbar_expect_tx(&sm.gfull[q], GBYTES);
            bulk_g2s(&sm.g[q][0], gsrc, GBYTES, &sm.gfull[q], pol_g);
            gsrc += EPB * SLAB;
            if (++gk == P) { gk = 0; gsrc += gjump; }
            --gleft;
        }
        if (UBULK && nmine > 1) issue_u(1);
    }
    DRows<T, P> dr;
    dr.init_shared(sm.D, i, j);
    T partial = T(0);
    T rg_r = T(0), rg_s = T(0), rg_W = T(0);       // RG: this thread's (r, s) = (xi_i, xi_j) and rho_i rho_j
    if constexpr (RG) { rg_r = sm.xr[i]; rg_s = sm.xr[j]; rg_W = sm.xr[P + i] * sm.xr[P + j]; }

    int q = 0;                 // ring stage of the slab being consumed
    uint32_t gphase = 0;       // its mbarrier parity
    T* wdst = w + ((int64_t)blockIdx.x * EPB + slot) * P3 + ij;
    const int64_t wstep = (int64_t)gridDim.x * (EPB * P3);
    int64_t grp = blockIdx.x;
    for (int64_t n = 0; n < nmine; ++n, grp += gridDim.x, wdst += wstep) {
        const bool ok = (FULL && EPB == 1) ? true : (lane_ok && grp * EPB + slot < E);
        const int ub = UBULK ? (int)(n & 1) : 0;
        const T* sue = &sm.u[ub][slot * P3];
        T uk[P], wk[P];
        if constexpr (UBULK) {
            mbar_wait(&sm.ufull[ub], (uint32_t)((n >> 1) & 1));
#pragma unroll
            for (int k = 0; k < P; ++k) { uk[k] = sue[k * P2 + ij]; wk[k] = T(0); }
        } else {
            // (every thread passed the barrier after part 1 of the previous group's last slab: its u is no longer read)
            const T* usrc = u + (grp * EPB + slot) * P3 + ij;
#pragma unroll
            for (int k = 0; k < P; ++k) {
                uk[k] = ok ? usrc[k * P2] : T(0);
                wk[k] = T(0);
                if (FULL || lane_ok) sm.u[0][slot * P3 + k * P2 + ij] = uk[k];
            }
            __syncthreads();
        }
        ColJac<T> cj;
        if constexpr (RG) col_jac_init<T>(vert + (grp * EPB + slot) * 24, ok, rg_r, rg_s, rg_W, cj);
#pragma unroll
        for (int k = 0; k < P; ++k) {
            const int buf = k & 1;
            T gr, gs;
            if constexpr (RG) {
                slab_part1_rg<T, P>(dp, dr, sue, uk, wk, cj, gl.xi[k], gl.rho[k], k, i, j, gr, gs);
            } else {
                mbar_wait(&sm.gfull[q], gphase);
                T g[6];
#pragma unroll
                for (int c = 0; c < 6; ++c) g[c] = sm.g[q][slot * SLAB + c * P2 + ij];
                slab_part1<T, P>(dp, dr, sue, uk, wk, g, k, i, j, gr, gs);
            }
            if (FULL || lane_ok) { sm.sgr[buf][slot * P2 + ij] = gr; sm.sgs[buf][slot * P2 + ij] = gs; }
            __syncthreads();
            // every thread has consumed stage q (and, on the last slab, this group's u buffer): refill
            if (tid == 0) {
                if (gleft > 0) {
                    mbar_expect_tx(&sm.gfull[q], GBYTES);
                    bulk_g2s(&sm.g[q][0], gsrc, GBYTES, &sm.gfull[q], pol_g);
                    gsrc += EPB * SLAB;
                    if ((k + NS) % P == P - 1) gsrc += gjump;     // that was the last slab of its group
                    --gleft;
                }
                if (UBULK && k == P - 1 && n + 2 < nmine) issue_u(n + 2);
            }
            wk[k] += slab_part2<T, P>(dr, i, j, &sm.sgr[buf][slot * P2], &sm.sgs[buf][slot * P2]);
            if (++q == NS) { q = 0; gphase ^= 1u; }
        }
        if (ok) {
#pragma unroll
            for (int k = 0; k < P; ++k) {
                T v = wk[k];
                if (Bm) v += lambda * Bm[(wdst - w) + k * P2] * uk[k];
                wdst[k * P2] = v;
                partial += uk[k] * v;
            }
        }
    }
    if (dot_out) block_dot_flush(partial, dot_out);
}

// ---------------------------------------------------------------------------------------------------------------
// ax_pencil: p >= 8, one element per CTA -- a measured ALTERNATIVE to ax_stream (sem_set_variant 4; the default only
// where it won: FP32 p = 9, FP64 p = 12).  ax_stream gives thread (i, j) a k-column and keeps FOUR rows / columns of D
// in its registers (80 registers at p = 10 in FP64), reads 4p shared-memory values per node and plane, and synchronises
// the CTA once per plane: at p = 10 that is 166 registers, 12 warps per SM, 333 shared-memory wavefronts per plane
// (0.79 per cycle and SM: the shared-memory pipe) and 0.69 of the HBM roofline.
// Here every 1-D contraction is done by a thread that owns a whole PENCIL of p values along the contracted direction:
// p inputs, p outputs, p^2 FMAs whose D operands have compile-time indices (uniform registers fed from the constant
// bank; no per-thread rows of D).  Per element:
//   A   thread (k, j): u_r along i for its row -> R;  thread (k, i): u_s along j for its column -> S          | barrier
//   B   thread (j, i): u_t along k in registers; per plane k: G from the slab ring, (g_r, g_s, g_t) = G (u_r, u_s, u_t),
//       g_r, g_s overwrite R, S in place, g_t stays in registers; then w_t = D^T g_t in registers         | barrier
//   C1  thread (k, j): D^T g_r along its row, in place in R                                                  | barrier
//   C2  thread (k, i): D^T g_s along its column, added into R                                                | barrier
//   C3  thread (j, i): w = w_t + R (+ lambda B u) -> global, fused dot                                       | barrier
// 20 shared-memory accesses per node instead of 48 (ncu at p = 10: 29.7 M wavefronts against 46.0 M), 5 CTA barriers
// per element instead of p, 128 registers.  The G slabs are released by a second ("empty") mbarrier per ring stage on
// which every thread arrives after its loads, so phase B has no CTA barrier; thread 0 refills the previous stage.
// Measured (profiles/r2_sweep.md): no faster than ax_stream at p = 10, 11 in FP64 -- the uniform-register traffic for D
// (LDCU / R2UR / moves) adds 0.9 instructions per FMA, and phase B consumes the element's G in one burst, so the CTA
// waits for the ring (long-scoreboard and branch stalls on the full barriers) with only 16 warps per SM to hide it.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <typename T, int P>
__device__ __forceinline__ void store_row(T* __restrict__ ptr, const T (&v)[P]) {
    if constexpr ((P * sizeof(T)) % 16 == 0) {
        constexpr int V = 16 / sizeof(T);
        using VT = typename std::conditional<sizeof(T) == 8, double2, float4>::type;
#pragma unroll
        for (int q = 0; q < P / V; ++q) {
            VT o;
            if constexpr (sizeof(T) == 8) { o.x = v[2 * q]; o.y = v[2 * q + 1]; }
            else { o.x = v[4 * q]; o.y = v[4 * q + 1]; o.z = v[4 * q + 2]; o.w = v[4 * q + 3]; }
            reinterpret_cast<VT*>(ptr)[q] = o;
        }
    } else if constexpr (sizeof(T) == 4 && (P * sizeof(T)) % 8 == 0) {
#pragma unroll
        for (int q = 0; q < P / 2; ++q) reinterpret_cast<float2*>(ptr)[q] = make_float2(v[2 * q], v[2 * q + 1]);
    } else {
#pragma unroll
        for (int l = 0; l < P; ++l) ptr[l] = v[l];
    }
}

// out[a] = sum_l D[a][l] in[l]  (TR = false)   or   sum_l D[l][a] in[l]  (TR = true); all D indices compile-time
template <typename T, int P, bool TR>
__device__ __forceinline__ void pencil_apply(const DParam<T, P>& dp, const T (&in)[P], T (&out)[P]) {
#pragma unroll
    for (int a = 0; a < P; ++a) {
        T acc = T(0);
#pragma unroll
        for (int l = 0; l < P; ++l) acc += (TR ? dp.D[l * P + a] : dp.D[a * P + l]) * in[l];
        out[a] = acc;
    }
}

template <typename T, int P, int NS>
struct PencilSmem {
    static constexpr int P2 = P * P, P3 = P2 * P;
    static constexpr int SLAB = 6 * P2 + ((6 * P2 * (int)sizeof(T)) % 16 ? 2 : 0);
    static constexpr bool UBULK = (P3 * (int)sizeof(T)) % 16 == 0;
    alignas(128) T g[NS][SLAB];
    alignas(128) T u[2][P3];
    alignas(16) T R[P3];
    alignas(16) T S[P3];
    alignas(8) uint64_t gfull[NS];
    alignas(8) uint64_t gempty[NS];
    alignas(8) uint64_t ufull[2];
};

template <typename T, int P, int NS, int MINB>
__global__ void __launch_bounds__(threads_of<P>(), MINB) ax_pencil(int64_t E, DParam<T, P> dp, const T* __restrict__ Gs,
                                                                   const T* __restrict__ Bm, T lambda,
                                                                   const T* __restrict__ u, T* __restrict__ w,
                                                                   const int* __restrict__ skip_flag,
                                                                   double* __restrict__ dot_out, int u_keep) {
    static_assert(epb_of<P>() == 1, "ax_pencil: one element per CTA");
    using SM = PencilSmem<T, P, NS>;
    constexpr int P2 = SM::P2, P3 = SM::P3, SLAB = SM::SLAB, NT = threads_of<P>();
    constexpr bool UBULK = SM::UBULK;
    constexpr uint32_t GBYTES = SLAB * sizeof(T), UBYTES = P3 * sizeof(T);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    SM& sm = *reinterpret_cast<SM*>(smem_raw);
    if (skip_flag && *skip_flag) return;
    const int tid = threadIdx.x;
    const bool act = tid < P2;
    const int64_t nmine = blockIdx.x < E ? (E - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;

    // producer state (thread 0): slabs in consumption order
    const T* gsrc = Gs + (int64_t)blockIdx.x * (P * SLAB);
    const int64_t gjump = (int64_t)(gridDim.x - 1) * (P * SLAB);
    int64_t gleft = nmine * P;
    int gk = 0;
    uint64_t pol_g = 0, pol_u = 0;
    auto issue_g = [&](int q) {
        mbar_expect_tx(&sm.gfull[q], GBYTES);
        bulk_g2s(&sm.g[q][0], gsrc, GBYTES, &sm.gfull[q], pol_g);
        gsrc += SLAB;
        if (++gk == P) { gk = 0; gsrc += gjump; }
        --gleft;
    };
    auto issue_u = [&](int64_t n) {
        const int b = (int)(n & 1);
        mbar_expect_tx(&sm.ufull[b], UBYTES);
        bulk_g2s(&sm.u[b][0], u + (blockIdx.x + n * gridDim.x) * P3, UBYTES, &sm.ufull[b], pol_u);
    };
    if (tid == 0) {
#pragma unroll
        for (int q = 0; q < NS; ++q) { mbar_init(&sm.gfull[q], 1); mbar_init(&sm.gempty[q], P2); }
        mbar_init(&sm.ufull[0], 1);
        mbar_init(&sm.ufull[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0 && nmine > 0) {
        pol_g = policy_evict_first();
        pol_u = u_keep ? policy_evict_last() : policy_evict_first();
        if (UBULK) issue_u(0);
        for (int q = 0; q < NS && gleft > 0; ++q) issue_g(q);
        if (UBULK && nmine > 1) issue_u(1);
    }
    int q = 0, pq = 0;                 // ring stage of the slab being consumed / of the previous one (thread 0)
    uint32_t gphase = 0, pphase = 0;
    bool have_prev = false;
    T partial = T(0);
    const int cb = (tid / P) * P2 + tid % P;       // column pencil (k, i) of this thread: base index, stride P
    for (int64_t n = 0; n < nmine; ++n) {
        const int64_t e = blockIdx.x + n * gridDim.x;
        const int ub = UBULK ? (int)(n & 1) : 0;
        T* su = &sm.u[ub][0];
        if constexpr (UBULK) {
            mbar_wait(&sm.ufull[ub], (uint32_t)((n >> 1) & 1));
        } else {
            for (int idx = tid; idx < P3; idx += NT) su[idx] = u[e * P3 + idx];
            __syncthreads();
        }
        T wt[P];
        if (act) {
            T in[P], out[P];
            load_row<T, P>(su + tid * P, in);                     // A: u_r for row (k, j) = tid
            pencil_apply<T, P, false>(dp, in, out);
            store_row<T, P>(&sm.R[tid * P], out);
#pragma unroll
            for (int l = 0; l < P; ++l) in[l] = su[cb + l * P];   // A: u_s for column (k, i)
            pencil_apply<T, P, false>(dp, in, out);
#pragma unroll
            for (int j = 0; j < P; ++j) sm.S[cb + j * P] = out[j];
        }
        __syncthreads();
        if (act) {
            T uk[P], gt[P];
#pragma unroll
            for (int k = 0; k < P; ++k) uk[k] = su[k * P2 + tid];
            pencil_apply<T, P, false>(dp, uk, gt);                // u_t along k
#pragma unroll
            for (int k = 0; k < P; ++k) {
                mbar_wait(&sm.gfull[q], gphase);
                T g[6];
#pragma unroll
                for (int c = 0; c < 6; ++c) g[c] = sm.g[q][c * P2 + tid];
                mbar_arrive(&sm.gempty[q]);
                if (tid == 0) {                                   // refill the stage of the previous slab
                    if (have_prev && gleft > 0) { mbar_wait(&sm.gempty[pq], pphase); issue_g(pq); }
                    pq = q; pphase = gphase; have_prev = true;
                }
                const T ur = sm.R[k * P2 + tid], us = sm.S[k * P2 + tid], ut = gt[k];
                sm.R[k * P2 + tid] = g[0] * ur + g[1] * us + g[2] * ut;
                sm.S[k * P2 + tid] = g[1] * ur + g[3] * us + g[4] * ut;
                gt[k] = g[2] * ur + g[4] * us + g[5] * ut;
                if (++q == NS) { q = 0; gphase ^= 1u; }
            }
            pencil_apply<T, P, true>(dp, gt, wt);                 // w_t = D^T g_t along k
        }
        __syncthreads();
        if (act) {                                                // C1: D^T g_r along the row, in place
            T in[P], out[P];
            load_row<T, P>(&sm.R[tid * P], in);
            pencil_apply<T, P, true>(dp, in, out);
            store_row<T, P>(&sm.R[tid * P], out);
        }
        __syncthreads();
        if (act) {                                                // C2: D^T g_s along the column, added into R
            T in[P], out[P];
#pragma unroll
            for (int l = 0; l < P; ++l) in[l] = sm.S[cb + l * P];
            pencil_apply<T, P, true>(dp, in, out);
#pragma unroll
            for (int j = 0; j < P; ++j) sm.R[cb + j * P] += out[j];
        }
        __syncthreads();
        if (act) {                                                // C3: results
            T* wdst = w + e * P3 + tid;
#pragma unroll
            for (int k = 0; k < P; ++k) {
                const T uu = su[k * P2 + tid];
                T v = wt[k] + sm.R[k * P2 + tid];
                if (Bm) v += lambda * Bm[e * P3 + k * P2 + tid] * uu;
                wdst[k * P2] = v;
                partial += uu * v;
            }
        }
        __syncthreads();                                          // R, S and this u buffer are free again
        if (UBULK && tid == 0 && n + 2 < nmine) issue_u(n + 2);
    }
    if (dot_out) block_dot_flush(partial, dot_out);
}

// ---------------------------------------------------------------------------------------------------------------
// ax_dmma: FP64, p = 8, ONE WARP per element; the r and s contractions of every k-plane run on the tensor cores as
// mma.sync.m8n8k4.f64 (DMMA).  north_star / SURVEY H3: "DMMA (m8n8k4 fits p = 8) only if measured faster" -- this is the
// kernel that measurement was made with, and it won (profiles/r2_dmma.md): it is the default for FP64 p = 8.  The DMMA rate of the part equals its DFMA
// rate, so the point is not flops: it is shared-memory wavefronts and issue slots.  Lane (g = lane / 4, t = lane % 4)
// owns the two columns (j = g, i = 2t, 2t + 1) of the element, which is exactly the C-fragment layout of m8n8k4, and
//   u_r = U_k D^T : A = the lane's own two u values (contraction index l = 2t + c for the two k-chunks c: a permutation
//                   of l shared by A and B, so no shuffle), B = constant fragment of D;
//   u_s = D U_k   : A = constant fragment of D, B = 2 values of the u plane read from shared memory;
//   w  += g_r D   : A = the lane's own two g_r values, B = constant;      w += D^T g_s : A = constant, B = 2 values of
//                   the g_s plane after one STS.128 + __syncwarp (the only exchange per plane);
//   the t direction stays in the lane's registers as in ax_stream.
// Per k-plane and element: 36 shared-memory wavefronts instead of 148, 8 DMMA + ~64 DFMA per lane instead of 2 x 126,
// no CTA barrier at all.  Streaming of G and u is the same mbarrier ring as ax_stream.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

template <int NS, int NU>
struct DmmaSmem {
    alignas(128) double g[NS][6 * 64];
    alignas(128) double u[NU][512];          // NU = 2: the next element's u lands while this one is worked on
    alignas(16) double sgs[2][64];
    alignas(8) uint64_t gfull[NS];
    alignas(8) uint64_t ufull[NU];
    alignas(16) double D[64];
};

template <int NS, int MINB, int NU>
__global__ void __launch_bounds__(32, MINB) ax_dmma(int64_t E, DParam<double, 8> dp, const double* __restrict__ Gs,
                                                    const double* __restrict__ Bm, double lambda,
                                                    const double* __restrict__ u, double* __restrict__ w,
                                                    const int* __restrict__ skip_flag, double* __restrict__ dot_out,
                                                    int u_keep) {
    using SM = DmmaSmem<NS, NU>;
    constexpr int P = 8, P2 = 64, P3 = 512, SLAB = 6 * 64;
    constexpr uint32_t GBYTES = SLAB * sizeof(double), UBYTES = P3 * sizeof(double);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    SM& sm = *reinterpret_cast<SM*>(smem_raw);
    if (skip_flag && *skip_flag) return;
    const int lane = threadIdx.x, g = lane >> 2, t = lane & 3;
    const int64_t nmine = blockIdx.x < E ? (E - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;

    const double* gsrc = Gs + (int64_t)blockIdx.x * (P * SLAB);
    const int64_t gjump = (int64_t)(gridDim.x - 1) * (P * SLAB);
    int64_t gleft = nmine * P;
    uint64_t pol_g = 0, pol_u = 0;
    auto issue_u = [&](int64_t n) {
        const int64_t e = blockIdx.x + n * gridDim.x;
        const int b = (int)(n % NU);
        mbar_expect_tx(&sm.ufull[b], UBYTES);
        bulk_g2s(&sm.u[b][0], u + e * P3, UBYTES, &sm.ufull[b], pol_u);
    };
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < NS; ++q) mbar_init(&sm.gfull[q], 1);
#pragma unroll
        for (int q = 0; q < NU; ++q) mbar_init(&sm.ufull[q], 1);
        mbar_fence_init();
    }
    sm.D[lane] = dp.D[lane];
    sm.D[lane + 32] = dp.D[lane + 32];
    __syncwarp();
    if (lane == 0 && nmine > 0) {
        pol_g = policy_evict_first();
        pol_u = u_keep ? policy_evict_last() : policy_evict_first();
        issue_u(0);
        int gk = 0;
        for (int q = 0; q < NS && gleft > 0; ++q) {
            mbar_expect_tx(&sm.gfull[q], GBYTES);
            bulk_g2s(&sm.g[q][0], gsrc, GBYTES, &sm.gfull[q], pol_g);
            gsrc += SLAB;
            if (++gk == P) { gk = 0; gsrc += gjump; }
            --gleft;
        }
        if (NU == 2 && nmine > 1) issue_u(1);
    }
    // constant fragments of D (volatile loads: pinned in registers, see DRows::init_shared)
    double Br[2], As[2], BrT[2], AsT[2];
    {
        const uint32_t base = smem_u32(sm.D);
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            Br[c] = DRows<double, 8>::lds_volatile(base + (uint32_t)((g * 8 + 2 * t + c) * 8));      // D[i=g][l=2t+c]
            As[c] = DRows<double, 8>::lds_volatile(base + (uint32_t)((g * 8 + 4 * c + t) * 8));      // D[j=g][l=4c+t]
            BrT[c] = DRows<double, 8>::lds_volatile(base + (uint32_t)(((2 * t + c) * 8 + g) * 8));   // D[l=2t+c][i=g]
            AsT[c] = DRows<double, 8>::lds_volatile(base + (uint32_t)(((4 * c + t) * 8 + g) * 8));   // D[l=4c+t][j=g]
        }
    }
    double partial = 0.0;
    int q = 0;
    uint32_t gphase = 0;
    const int own = g * 8 + 2 * t;                     // the lane's two nodes (j = g, i = 2t, 2t+1) inside a plane
    double* wdst = w + (int64_t)blockIdx.x * P3 + own;
    const int64_t wstep = (int64_t)gridDim.x * P3;
    for (int64_t n = 0; n < nmine; ++n, wdst += wstep) {
        const int ub = (int)(n % NU);
        mbar_wait(&sm.ufull[ub], (uint32_t)((n / NU) & 1));
        const double* sue = &sm.u[ub][0];
        double uk[P][2], wk[P][2];
#pragma unroll
        for (int k = 0; k < P; ++k) {
            const double2 v = *reinterpret_cast<const double2*>(sue + k * P2 + own);
            uk[k][0] = v.x; uk[k][1] = v.y; wk[k][0] = 0.0; wk[k][1] = 0.0;
        }
#pragma unroll
        for (int k = 0; k < P; ++k) {
            mbar_wait(&sm.gfull[q], gphase);
            double G6[6][2];
#pragma unroll
            for (int c = 0; c < 6; ++c) {
                const double2 v = *reinterpret_cast<const double2*>(&sm.g[q][c * P2 + own]);
                G6[c][0] = v.x; G6[c][1] = v.y;
            }
            // u_r = U_k D^T  and  u_s = D U_k  on the tensor cores
            double ur[2] = {0.0, 0.0}, us[2] = {0.0, 0.0};
            dmma884(ur[0], ur[1], uk[k][0], Br[0]);
            dmma884(us[0], us[1], As[0], sue[k * P2 + t * P + g]);
            dmma884(ur[0], ur[1], uk[k][1], Br[1]);
            dmma884(us[0], us[1], As[1], sue[k * P2 + (4 + t) * P + g]);
            double ut[2] = {0.0, 0.0};
#pragma unroll
            for (int l = 0; l < P; ++l) { ut[0] += dp.D[k * P + l] * uk[l][0]; ut[1] += dp.D[k * P + l] * uk[l][1]; }
            double gr[2], gs[2], gt[2];
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                gr[b] = G6[0][b] * ur[b] + G6[1][b] * us[b] + G6[2][b] * ut[b];
                gs[b] = G6[1][b] * ur[b] + G6[3][b] * us[b] + G6[4][b] * ut[b];
                gt[b] = G6[2][b] * ur[b] + G6[4][b] * us[b] + G6[5][b] * ut[b];
            }
            const int buf = k & 1;
            *reinterpret_cast<double2*>(&sm.sgs[buf][own]) = make_double2(gs[0], gs[1]);
#pragma unroll
            for (int l = 0; l < P; ++l) { wk[l][0] += dp.D[k * P + l] * gt[0]; wk[l][1] += dp.D[k * P + l] * gt[1]; }
            __syncwarp();
            // every lane has consumed stage q (and, on the last plane, this element's u buffer): refill
            if (lane == 0) {
                if (gleft > 0) {
                    mbar_expect_tx(&sm.gfull[q], GBYTES);
                    bulk_g2s(&sm.g[q][0], gsrc, GBYTES, &sm.gfull[q], pol_g);
                    gsrc += SLAB;
                    if ((k + NS) % P == P - 1) gsrc += gjump;
                    --gleft;
                }
                if (k == P - 1 && n + NU < nmine) issue_u(n + NU);
            }
            // w_k += g_r D + D^T g_s
            double a0[2] = {0.0, 0.0}, a1[2] = {0.0, 0.0};
            dmma884(a0[0], a0[1], gr[0], BrT[0]);
            dmma884(a1[0], a1[1], AsT[0], sm.sgs[buf][t * P + g]);
            dmma884(a0[0], a0[1], gr[1], BrT[1]);
            dmma884(a1[0], a1[1], AsT[1], sm.sgs[buf][(4 + t) * P + g]);
            wk[k][0] += a0[0] + a1[0];
            wk[k][1] += a0[1] + a1[1];
            if (++q == NS) { q = 0; gphase ^= 1u; }
        }
#pragma unroll
        for (int k = 0; k < P; ++k) {
            double v0 = wk[k][0], v1 = wk[k][1];
            if (Bm) {
                const double2 bm = *reinterpret_cast<const double2*>(Bm + (wdst - w) + k * P2);
                v0 += lambda * bm.x * uk[k][0];
                v1 += lambda * bm.y * uk[k][1];
            }
            *reinterpret_cast<double2*>(wdst + k * P2) = make_double2(v0, v1);
            partial += uk[k][0] * v0 + uk[k][1] * v1;
        }
    }
    if (dot_out) {
        for (int o = 16; o; o >>= 1) partial += __shfl_xor_sync(0xffffffffu, partial, o);
        if (lane == 0) atomicAdd(dot_out, partial);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// ax_dmma_rg: a9 (north_star: "recomputed geometric factors to cut bytes per node"), FP64, p = 8, trilinear elements.
// The tensor-core kernel above without the G ring: the six factors of a node are recomputed in registers from the
// element's 8 vertices (192 bytes, bulk-copied beside u) -- 16 bytes per node of HBM traffic instead of 64, about
// twice the FP64 arithmetic (the 3 x 3 Jacobian of the trilinear map is linear in t for fixed (r, s), so a lane keeps
// 24 coefficients for its two columns and a plane costs 6 FMAs for J, then the adjugate, one division and
// G = (W / det) adj adj^T: ~65 FMA-pipe instructions per node against ~57 for the whole rest of the operator).
// The kernel is bound by the FP64 pipe, not by memory; it replaces ax_simple<RECOMP> for p = 8.
// lambda B u is accumulated plane by plane (B = W det comes out of the same computation).
// ---------------------------------------------------------------------------------------------------------------
struct GllP8 { double xi[8], rho[8]; };

template <int NU>
struct DmmaRgSmem {
    alignas(128) double u[NU][512];
    alignas(16) double vert[NU][24];
    alignas(16) double sgs[2][64];
    alignas(8) uint64_t ufull[NU];
    alignas(16) double D[64];
    alignas(16) double xr[16];               // xi, rho for lane-dependent indices (a by-value parameter indexed
};                                           // dynamically would be copied to local memory)

template <int MINB, int NU, bool HELM>
__global__ void __launch_bounds__(32, MINB) ax_dmma_rg(int64_t E, DParam<double, 8> dp, GllP8 gll,
                                                       const double* __restrict__ vert, double lambda,
                                                       const double* __restrict__ u, double* __restrict__ w,
                                                       const int* __restrict__ skip_flag, double* __restrict__ dot_out,
                                                       int u_keep) {
    using SM = DmmaRgSmem<NU>;
    constexpr int P = 8, P2 = 64, P3 = 512;
    constexpr uint32_t UBYTES = P3 * sizeof(double), VBYTES = 24 * sizeof(double);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    SM& sm = *reinterpret_cast<SM*>(smem_raw);
    if (skip_flag && *skip_flag) return;
    const int lane = threadIdx.x, g = lane >> 2, t = lane & 3;
    const int64_t nmine = blockIdx.x < E ? (E - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    uint64_t pol_u = 0, pol_v = 0;
    auto issue_u = [&](int64_t n) {
        const int64_t e = blockIdx.x + n * gridDim.x;
        const int b = (int)(n % NU);
        mbar_expect_tx(&sm.ufull[b], UBYTES + VBYTES);
        bulk_g2s(&sm.u[b][0], u + e * P3, UBYTES, &sm.ufull[b], pol_u);
        bulk_g2s(&sm.vert[b][0], vert + e * 24, VBYTES, &sm.ufull[b], pol_v);
    };
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < NU; ++q) mbar_init(&sm.ufull[q], 1);
        mbar_fence_init();
    }
    sm.D[lane] = dp.D[lane];
    sm.D[lane + 32] = dp.D[lane + 32];
#pragma unroll
    for (int q = 0; q < 8; ++q)
        if (lane == q) { sm.xr[q] = gll.xi[q]; sm.xr[8 + q] = gll.rho[q]; }
    __syncwarp();
    if (lane == 0 && nmine > 0) {
        pol_v = policy_evict_first();
        pol_u = u_keep ? policy_evict_last() : policy_evict_first();
        issue_u(0);
        if (NU == 2 && nmine > 1) issue_u(1);
    }
    double Br[2], As[2], BrT[2], AsT[2];
    {
        const uint32_t base = smem_u32(sm.D);
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            Br[c] = DRows<double, 8>::lds_volatile(base + (uint32_t)((g * 8 + 2 * t + c) * 8));
            As[c] = DRows<double, 8>::lds_volatile(base + (uint32_t)((g * 8 + 4 * c + t) * 8));
            BrT[c] = DRows<double, 8>::lds_volatile(base + (uint32_t)(((2 * t + c) * 8 + g) * 8));
            AsT[c] = DRows<double, 8>::lds_volatile(base + (uint32_t)(((4 * c + t) * 8 + g) * 8));
        }
    }
    // the lane's two columns: (r, s) = (xi_i, xi_j), i = 2t, 2t + 1, j = g; W_ij = rho_i rho_j
    const double sj = sm.xr[g], rj = sm.xr[8 + g];
    const double ri[2] = {sm.xr[2 * t], sm.xr[2 * t + 1]};
    const double Wij[2] = {sm.xr[8 + 2 * t] * rj, sm.xr[8 + 2 * t + 1] * rj};
    double partial = 0.0;
    const int own = g * 8 + 2 * t;
    double* wdst = w + (int64_t)blockIdx.x * P3 + own;
    const int64_t wstep = (int64_t)gridDim.x * P3;
    for (int64_t n = 0; n < nmine; ++n, wdst += wstep) {
        const int ub = (int)(n % NU);
        mbar_wait(&sm.ufull[ub], (uint32_t)((n / NU) & 1));
        const double* sue = &sm.u[ub][0];
        // Jacobian coefficients of the lane's two columns: dx/dr = Ja + Jb t, dx/ds = Jc + Jd t, dx/dt = Je (S5)
        double Ja[3], Jb[3], Jc[2][3], Jd[2][3], Je[2][3];
        {
            double X[8][3], cf[8][3];
#pragma unroll
            for (int v = 0; v < 8; ++v)
#pragma unroll
                for (int d = 0; d < 3; ++d) X[v][d] = sm.vert[ub][v * 3 + d];
            sem_trilinear_coef(X, cf);
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                Ja[d] = cf[1][d] + cf[4][d] * sj;
                Jb[d] = cf[5][d] + cf[7][d] * sj;
#pragma unroll
                for (int b = 0; b < 2; ++b) {
                    Jc[b][d] = cf[2][d] + cf[4][d] * ri[b];
                    Jd[b][d] = cf[6][d] + cf[7][d] * ri[b];
                    Je[b][d] = cf[3][d] + cf[5][d] * ri[b] + (cf[6][d] + cf[7][d] * ri[b]) * sj;
                }
            }
        }
        double uk[P][2], wk[P][2];
#pragma unroll
        for (int k = 0; k < P; ++k) {
            const double2 v = *reinterpret_cast<const double2*>(sue + k * P2 + own);
            uk[k][0] = v.x; uk[k][1] = v.y; wk[k][0] = 0.0; wk[k][1] = 0.0;
        }
#pragma unroll
        for (int k = 0; k < P; ++k) {
            const double tk = gll.xi[k], rk = gll.rho[k];
            double ur[2] = {0.0, 0.0}, us[2] = {0.0, 0.0};
            dmma884(ur[0], ur[1], uk[k][0], Br[0]);
            dmma884(us[0], us[1], As[0], sue[k * P2 + t * P + g]);
            dmma884(ur[0], ur[1], uk[k][1], Br[1]);
            dmma884(us[0], us[1], As[1], sue[k * P2 + (4 + t) * P + g]);
            double ut[2] = {0.0, 0.0};
#pragma unroll
            for (int l = 0; l < P; ++l) { ut[0] += dp.D[k * P + l] * uk[l][0]; ut[1] += dp.D[k * P + l] * uk[l][1]; }
            // G (u_r, u_s, u_t) without forming G:  G = (W / det) A A^T with the adjugate rows a_0 = x_s x x_t,
            // a_1 = x_t x x_r, a_2 = x_r x x_s of the Jacobian columns, so  G v = (W / det) A (A^T v): 21 FMAs
            // instead of 24 for G plus 9 for the product; det = x_r . a_0; one reciprocal
            double gr[2], gs[2], gt[2], Bk[2];
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                double xr[3], xs[3];
#pragma unroll
                for (int d = 0; d < 3; ++d) { xr[d] = Ja[d] + Jb[d] * tk; xs[d] = Jc[b][d] + Jd[b][d] * tk; }
                const double* xt = Je[b];
                const double a0x = xs[1] * xt[2] - xs[2] * xt[1], a0y = xs[2] * xt[0] - xs[0] * xt[2],
                             a0z = xs[0] * xt[1] - xs[1] * xt[0];
                const double a1x = xt[1] * xr[2] - xt[2] * xr[1], a1y = xt[2] * xr[0] - xt[0] * xr[2],
                             a1z = xt[0] * xr[1] - xt[1] * xr[0];
                const double a2x = xr[1] * xs[2] - xr[2] * xs[1], a2y = xr[2] * xs[0] - xr[0] * xs[2],
                             a2z = xr[0] * xs[1] - xr[1] * xs[0];
                const double det = xr[0] * a0x + xr[1] * a0y + xr[2] * a0z;
                const double Wk = Wij[b] * rk;
                const double sc = Wk * __drcp_rn(det);
                const double zx = a0x * ur[b] + a1x * us[b] + a2x * ut[b];
                const double zy = a0y * ur[b] + a1y * us[b] + a2y * ut[b];
                const double zz = a0z * ur[b] + a1z * us[b] + a2z * ut[b];
                gr[b] = sc * (a0x * zx + a0y * zy + a0z * zz);
                gs[b] = sc * (a1x * zx + a1y * zy + a1z * zz);
                gt[b] = sc * (a2x * zx + a2y * zy + a2z * zz);
                Bk[b] = HELM ? lambda * Wk * det : 0.0;
            }
            const int buf = k & 1;
            *reinterpret_cast<double2*>(&sm.sgs[buf][own]) = make_double2(gs[0], gs[1]);
#pragma unroll
            for (int l = 0; l < P; ++l) { wk[l][0] += dp.D[k * P + l] * gt[0]; wk[l][1] += dp.D[k * P + l] * gt[1]; }
            __syncwarp();
            double a0[2] = {0.0, 0.0}, a1[2] = {0.0, 0.0};
            dmma884(a0[0], a0[1], gr[0], BrT[0]);
            dmma884(a1[0], a1[1], AsT[0], sm.sgs[buf][t * P + g]);
            dmma884(a0[0], a0[1], gr[1], BrT[1]);
            dmma884(a1[0], a1[1], AsT[1], sm.sgs[buf][(4 + t) * P + g]);
            wk[k][0] += a0[0] + a1[0];
            wk[k][1] += a0[1] + a1[1];
            if constexpr (HELM) { wk[k][0] += Bk[0] * uk[k][0]; wk[k][1] += Bk[1] * uk[k][1]; }
        }
        // every lane has read this element's u (the last plane's B operands before the __syncwarp above): refill
        __syncwarp();
        if (lane == 0 && n + NU < nmine) issue_u(n + NU);
#pragma unroll
        for (int k = 0; k < P; ++k) {
            *reinterpret_cast<double2*>(wdst + k * P2) = make_double2(wk[k][0], wk[k][1]);
            partial += uk[k][0] * wk[k][0] + uk[k][1] * wk[k][1];
        }
    }
    if (dot_out) {
        for (int o = 16; o; o >>= 1) partial += __shfl_xor_sync(0xffffffffu, partial, o);
        if (lane == 0) atomicAdd(dot_out, partial);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// ax_tf32: FP32, p = 8, one warp per element like ax_dmma, the r and s contractions on the tensor cores as
// mma.sync.m16n8k8 TF32 in THREE passes (x = hi + lo with hi = tf32(x), lo = tf32(x - hi); hi*hi + lo*hi + hi*lo, the
// dropped lo*lo term is 2^-22 relative: FP32-level accuracy, inside the 1e-5 bar of S16; accumulation in FP32).  There
// is no exact single-pass FP32 tensor-core path (TF32 carries 10 mantissa bits).  The scalar FP32 kernel issues the same
// shared-memory traffic as the FP64 one for half the bytes and sits at 0.71 of the HBM roofline; here two k-planes share
// one MMA in the r direction (M = 16 = two planes of 8 rows; the lane's own four values are its A fragment through the
// same permuted contraction index as in ax_dmma), the s direction takes one MMA per plane with D in the upper half of A.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void split_tf32(float x, uint32_t& hi, uint32_t& lo) {
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(hi) : "f"(x));
    const float rest = x - __uint_as_float(hi);
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(lo) : "f"(rest));
}
__device__ __forceinline__ void mma1688(float (&d)[4], const uint32_t (&a)[4], const uint32_t (&b)[2]) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}
// d += a * b in three TF32 passes; the operands arrive already split
__device__ __forceinline__ void mma3(float (&d)[4], const uint32_t (&ah)[4], const uint32_t (&al)[4],
                                     const uint32_t (&bh)[2], const uint32_t (&bl)[2]) {
    mma1688(d, al, bh);
    mma1688(d, ah, bl);
    mma1688(d, ah, bh);
}

template <int NS>
struct Tf32Smem {
    alignas(128) float g[NS][2][6 * 64];        // a stage = the slabs of two consecutive planes: one bulk copy of 3 KB
    alignas(128) float u[2][512];
    alignas(16) float sgs[2][2][64];            // [buffer][plane of the pair][j * 8 + i]
    alignas(8) uint64_t gfull[NS];
    alignas(8) uint64_t ufull[2];
    alignas(16) float D[64];
};

template <int NS, int MINB>
__global__ void __launch_bounds__(32, MINB) ax_tf32(int64_t E, DParam<float, 8> dp, const float* __restrict__ Gs,
                                                    const float* __restrict__ Bm, float lambda,
                                                    const float* __restrict__ u, float* __restrict__ w,
                                                    const int* __restrict__ skip_flag, double* __restrict__ dot_out,
                                                    int u_keep) {
    using SM = Tf32Smem<NS>;
    constexpr int P = 8, P2 = 64, P3 = 512, SLAB = 6 * 64;
    constexpr uint32_t GBYTES = 2 * SLAB * sizeof(float), UBYTES = P3 * sizeof(float);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    SM& sm = *reinterpret_cast<SM*>(smem_raw);
    if (skip_flag && *skip_flag) return;
    const int lane = threadIdx.x, g = lane >> 2, t = lane & 3;
    const int64_t nmine = blockIdx.x < E ? (E - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;

    const float* gsrc = Gs + (int64_t)blockIdx.x * (P * SLAB);
    const int64_t gjump = (int64_t)(gridDim.x - 1) * (P * SLAB);
    int64_t gleft = nmine * (P / 2);                  // plane pairs still to issue
    int gk = 0;                                       // pair index (within its element) of the next one
    uint64_t pol_g = 0, pol_u = 0;
    auto issue_u = [&](int64_t n) {
        const int64_t e = blockIdx.x + n * gridDim.x;
        const int b = (int)(n & 1);
        mbar_expect_tx(&sm.ufull[b], UBYTES);
        bulk_g2s(&sm.u[b][0], u + e * P3, UBYTES, &sm.ufull[b], pol_u);
    };
    auto issue_g = [&](int stage) {
        mbar_expect_tx(&sm.gfull[stage], GBYTES);
        bulk_g2s(&sm.g[stage][0][0], gsrc, GBYTES, &sm.gfull[stage], pol_g);
        gsrc += 2 * SLAB;
        if (++gk == P / 2) { gk = 0; gsrc += gjump; }
        --gleft;
    };
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < NS; ++q) mbar_init(&sm.gfull[q], 1);
        mbar_init(&sm.ufull[0], 1);
        mbar_init(&sm.ufull[1], 1);
        mbar_fence_init();
    }
    sm.D[lane] = dp.D[lane];
    sm.D[lane + 32] = dp.D[lane + 32];
    __syncwarp();
    if (lane == 0 && nmine > 0) {
        pol_g = policy_evict_first();
        pol_u = u_keep ? policy_evict_last() : policy_evict_first();
        issue_u(0);
        for (int q = 0; q < NS && gleft > 0; ++q) issue_g(q);
        if (nmine > 1) issue_u(1);
    }
    // constant fragments of D, split once: B of the r contractions, A (rows 0-7; rows 8-15 zero) of the s contractions
    uint32_t Brh[2], Brl[2], BrTh[2], BrTl[2], Ash[4], Asl[4], AsTh[4], AsTl[4];
    {
        const uint32_t base = smem_u32(sm.D);
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            split_tf32(DRows<float, 8>::lds_volatile(base + (uint32_t)((g * 8 + 2 * t + c) * 4)), Brh[c], Brl[c]);     // D[i=g][l=2t+c]
            split_tf32(DRows<float, 8>::lds_volatile(base + (uint32_t)(((2 * t + c) * 8 + g) * 4)), BrTh[c], BrTl[c]); // D[l=2t+c][i=g]
            split_tf32(DRows<float, 8>::lds_volatile(base + (uint32_t)((g * 8 + 4 * c + t) * 4)), Ash[2 * c], Asl[2 * c]);     // D[j=g][l=4c+t]
            split_tf32(DRows<float, 8>::lds_volatile(base + (uint32_t)(((4 * c + t) * 8 + g) * 4)), AsTh[2 * c], AsTl[2 * c]); // D[l=4c+t][j=g]
            Ash[2 * c + 1] = Asl[2 * c + 1] = AsTh[2 * c + 1] = AsTl[2 * c + 1] = 0u;
        }
    }
    float partial = 0.f;
    int q = 0;
    uint32_t gphase = 0;
    const int own = g * 8 + 2 * t;
    float* wdst = w + (int64_t)blockIdx.x * P3 + own;
    const int64_t wstep = (int64_t)gridDim.x * P3;
    for (int64_t n = 0; n < nmine; ++n, wdst += wstep) {
        const int ub = (int)(n & 1);
        mbar_wait(&sm.ufull[ub], (uint32_t)((n >> 1) & 1));
        const float* sue = &sm.u[ub][0];
        float uk[P][2], wk[P][2];
#pragma unroll
        for (int k = 0; k < P; ++k) {
            const float2 v = *reinterpret_cast<const float2*>(sue + k * P2 + own);
            uk[k][0] = v.x; uk[k][1] = v.y; wk[k][0] = 0.f; wk[k][1] = 0.f;
        }
#pragma unroll
        for (int k = 0; k < P; k += 2) {
            mbar_wait(&sm.gfull[q], gphase);
            // u_r of both planes in one MMA: A = the lane's own four values
            float ur[4] = {0.f, 0.f, 0.f, 0.f};
            {
                uint32_t ah[4], al[4];
                split_tf32(uk[k][0], ah[0], al[0]);
                split_tf32(uk[k + 1][0], ah[1], al[1]);
                split_tf32(uk[k][1], ah[2], al[2]);
                split_tf32(uk[k + 1][1], ah[3], al[3]);
                mma3(ur, ah, al, Brh, Brl);
            }
            float gr[2][2], gt[2][2];
            const int buf = (k >> 1) & 1;
#pragma unroll
            for (int h = 0; h < 2; ++h) {                       // the two planes of the pair
                const int kk = k + h;
                float us4[4] = {0.f, 0.f, 0.f, 0.f};
                {
                    uint32_t bh[2], bl[2];
                    split_tf32(sue[kk * P2 + t * P + g], bh[0], bl[0]);
                    split_tf32(sue[kk * P2 + (4 + t) * P + g], bh[1], bl[1]);
                    mma3(us4, Ash, Asl, bh, bl);
                }
                float ut[2] = {0.f, 0.f};
#pragma unroll
                for (int l = 0; l < P; ++l) { ut[0] += dp.D[kk * P + l] * uk[l][0]; ut[1] += dp.D[kk * P + l] * uk[l][1]; }
                float G6[6][2];
#pragma unroll
                for (int c = 0; c < 6; ++c) {
                    const float2 v = *reinterpret_cast<const float2*>(&sm.g[q][h][c * P2 + own]);
                    G6[c][0] = v.x; G6[c][1] = v.y;
                }
                float gs[2];
#pragma unroll
                for (int b = 0; b < 2; ++b) {
                    const float r_ = ur[2 * h + b], s_ = us4[b], t_ = ut[b];
                    gr[h][b] = G6[0][b] * r_ + G6[1][b] * s_ + G6[2][b] * t_;
                    gs[b] = G6[1][b] * r_ + G6[3][b] * s_ + G6[4][b] * t_;
                    gt[h][b] = G6[2][b] * r_ + G6[4][b] * s_ + G6[5][b] * t_;
                }
                *reinterpret_cast<float2*>(&sm.sgs[buf][h][own]) = make_float2(gs[0], gs[1]);
#pragma unroll
                for (int l = 0; l < P; ++l) { wk[l][0] += dp.D[kk * P + l] * gt[h][0]; wk[l][1] += dp.D[kk * P + l] * gt[h][1]; }
            }
            __syncwarp();
            if (lane == 0) {                                    // the stage is consumed by every lane: refill
                if (gleft > 0) issue_g(q);
                if (k == P - 2 && n + 2 < nmine) issue_u(n + 2);
            }
            // w += g_r D (both planes, one MMA) + D^T g_s (one MMA per plane)
            float ar[4] = {0.f, 0.f, 0.f, 0.f};
            {
                uint32_t ah[4], al[4];
                split_tf32(gr[0][0], ah[0], al[0]);
                split_tf32(gr[1][0], ah[1], al[1]);
                split_tf32(gr[0][1], ah[2], al[2]);
                split_tf32(gr[1][1], ah[3], al[3]);
                mma3(ar, ah, al, BrTh, BrTl);
            }
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                float as4[4] = {0.f, 0.f, 0.f, 0.f};
                uint32_t bh[2], bl[2];
                split_tf32(sm.sgs[buf][h][t * P + g], bh[0], bl[0]);
                split_tf32(sm.sgs[buf][h][(4 + t) * P + g], bh[1], bl[1]);
                mma3(as4, AsTh, AsTl, bh, bl);
                wk[k + h][0] += ar[2 * h] + as4[0];
                wk[k + h][1] += ar[2 * h + 1] + as4[1];
            }
            if (++q == NS) { q = 0; gphase ^= 1u; }
        }
#pragma unroll
        for (int k = 0; k < P; ++k) {
            float v0 = wk[k][0], v1 = wk[k][1];
            if (Bm) {
                const float2 bm = *reinterpret_cast<const float2*>(Bm + (wdst - w) + k * P2);
                v0 += lambda * bm.x * uk[k][0];
                v1 += lambda * bm.y * uk[k][1];
            }
            *reinterpret_cast<float2*>(wdst + k * P2) = make_float2(v0, v1);
            partial += uk[k][0] * v0 + uk[k][1] * v1;
        }
    }
    if (dot_out) {
        double v = (double)partial;
        for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) atomicAdd(dot_out, v);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// ax_dmma_many: the same operator applied to NF fields that share the geometric factors (NEXT-4: "3 Helmholtz problems --
// one for each velocity component"): G is streamed ONCE per element and k-plane and used for all NF fields, so the
// compulsory traffic is 48 + 16 NF bytes per node instead of 64 NF (NF = 3: 96 instead of 192).  One warp per element
// as in ax_dmma; the w accumulators of all fields stay in registers (NF x 16 doubles), the u columns are re-read from
// shared memory plane by plane (they cannot stay in registers as well).  Field f lives at u + f * stride, w + f * stride.
// ---------------------------------------------------------------------------------------------------------------
template <int NF, int NS>
struct DmmaManySmem {
    alignas(128) double g[NS][6 * 64];
    alignas(128) double u[NF][512];
    alignas(16) double sgs[2][64];
    alignas(8) uint64_t gfull[NS];
    alignas(8) uint64_t ufull;
    alignas(16) double D[64];
};

template <int NF, int NS, int MINB>
__global__ void __launch_bounds__(32, MINB) ax_dmma_many(int64_t E, DParam<double, 8> dp, const double* __restrict__ Gs,
                                                         const double* __restrict__ Bm, double lambda,
                                                         const double* __restrict__ u, double* __restrict__ w,
                                                         int64_t stride, const int* __restrict__ skip_flag,
                                                         double* __restrict__ dot_out, int64_t dot_stride, int u_keep) {
    using SM = DmmaManySmem<NF, NS>;
    constexpr int P = 8, P2 = 64, P3 = 512, SLAB = 6 * 64;
    constexpr uint32_t GBYTES = SLAB * sizeof(double), UBYTES = P3 * sizeof(double);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    SM& sm = *reinterpret_cast<SM*>(smem_raw);
    if (skip_flag && *skip_flag) return;
    const int lane = threadIdx.x, g = lane >> 2, t = lane & 3;
    const int64_t nmine = blockIdx.x < E ? (E - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;

    const double* gsrc = Gs + (int64_t)blockIdx.x * (P * SLAB);
    const int64_t gjump = (int64_t)(gridDim.x - 1) * (P * SLAB);
    int64_t gleft = nmine * P;
    uint64_t pol_g = 0, pol_u = 0;
    auto issue_u = [&](int64_t n) {                      // the NF element blocks of u: one barrier phase per element
        const int64_t e = blockIdx.x + n * gridDim.x;
        mbar_expect_tx(&sm.ufull, NF * UBYTES);
#pragma unroll
        for (int f = 0; f < NF; ++f) bulk_g2s(&sm.u[f][0], u + f * stride + e * P3, UBYTES, &sm.ufull, pol_u);
    };
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < NS; ++q) mbar_init(&sm.gfull[q], 1);
        mbar_init(&sm.ufull, 1);
        mbar_fence_init();
    }
    sm.D[lane] = dp.D[lane];
    sm.D[lane + 32] = dp.D[lane + 32];
    __syncwarp();
    if (lane == 0 && nmine > 0) {
        pol_g = policy_evict_first();
        pol_u = u_keep ? policy_evict_last() : policy_evict_first();
        issue_u(0);
        int gk = 0;
        for (int q = 0; q < NS && gleft > 0; ++q) {
            mbar_expect_tx(&sm.gfull[q], GBYTES);
            bulk_g2s(&sm.g[q][0], gsrc, GBYTES, &sm.gfull[q], pol_g);
            gsrc += SLAB;
            if (++gk == P) { gk = 0; gsrc += gjump; }
            --gleft;
        }
    }
    double Br[2], As[2], BrT[2], AsT[2];
    {
        const uint32_t base = smem_u32(sm.D);
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            Br[c] = DRows<double, 8>::lds_volatile(base + (uint32_t)((g * 8 + 2 * t + c) * 8));
            As[c] = DRows<double, 8>::lds_volatile(base + (uint32_t)((g * 8 + 4 * c + t) * 8));
            BrT[c] = DRows<double, 8>::lds_volatile(base + (uint32_t)(((2 * t + c) * 8 + g) * 8));
            AsT[c] = DRows<double, 8>::lds_volatile(base + (uint32_t)(((4 * c + t) * 8 + g) * 8));
        }
    }
    double partial[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) partial[f] = 0.0;
    int q = 0;
    uint32_t gphase = 0;
    const int own = g * 8 + 2 * t;
    for (int64_t n = 0; n < nmine; ++n) {
        const int64_t e = blockIdx.x + n * gridDim.x;
        mbar_wait(&sm.ufull, (uint32_t)(n & 1));
        double wk[NF][P][2];
#pragma unroll
        for (int f = 0; f < NF; ++f)
#pragma unroll
            for (int k = 0; k < P; ++k) { wk[f][k][0] = 0.0; wk[f][k][1] = 0.0; }
#pragma unroll
        for (int k = 0; k < P; ++k) {
            mbar_wait(&sm.gfull[q], gphase);
            double G6[6][2];
#pragma unroll
            for (int c = 0; c < 6; ++c) {
                const double2 v = *reinterpret_cast<const double2*>(&sm.g[q][c * P2 + own]);
                G6[c][0] = v.x; G6[c][1] = v.y;
            }
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                const double* sue = &sm.u[f][0];
                double uk[P][2];
#pragma unroll
                for (int l = 0; l < P; ++l) {
                    const double2 v = *reinterpret_cast<const double2*>(sue + l * P2 + own);
                    uk[l][0] = v.x; uk[l][1] = v.y;
                }
                double ur[2] = {0.0, 0.0}, us[2] = {0.0, 0.0};
                dmma884(ur[0], ur[1], uk[k][0], Br[0]);
                dmma884(us[0], us[1], As[0], sue[k * P2 + t * P + g]);
                dmma884(ur[0], ur[1], uk[k][1], Br[1]);
                dmma884(us[0], us[1], As[1], sue[k * P2 + (4 + t) * P + g]);
                double ut[2] = {0.0, 0.0};
#pragma unroll
                for (int l = 0; l < P; ++l) { ut[0] += dp.D[k * P + l] * uk[l][0]; ut[1] += dp.D[k * P + l] * uk[l][1]; }
                double gr[2], gs[2], gt[2];
#pragma unroll
                for (int b = 0; b < 2; ++b) {
                    gr[b] = G6[0][b] * ur[b] + G6[1][b] * us[b] + G6[2][b] * ut[b];
                    gs[b] = G6[1][b] * ur[b] + G6[3][b] * us[b] + G6[4][b] * ut[b];
                    gt[b] = G6[2][b] * ur[b] + G6[4][b] * us[b] + G6[5][b] * ut[b];
                }
                const int buf = (k * NF + f) & 1;
                *reinterpret_cast<double2*>(&sm.sgs[buf][own]) = make_double2(gs[0], gs[1]);
#pragma unroll
                for (int l = 0; l < P; ++l) { wk[f][l][0] += dp.D[k * P + l] * gt[0]; wk[f][l][1] += dp.D[k * P + l] * gt[1]; }
                __syncwarp();
                if (f == NF - 1 && lane == 0 && gleft > 0) {      // every lane has consumed stage q for all fields: refill
                    mbar_expect_tx(&sm.gfull[q], GBYTES);
                    bulk_g2s(&sm.g[q][0], gsrc, GBYTES, &sm.gfull[q], pol_g);
                    gsrc += SLAB;
                    if ((k + NS) % P == P - 1) gsrc += gjump;
                    --gleft;
                }
                double a0[2] = {0.0, 0.0}, a1[2] = {0.0, 0.0};
                dmma884(a0[0], a0[1], gr[0], BrT[0]);
                dmma884(a1[0], a1[1], AsT[0], sm.sgs[buf][t * P + g]);
                dmma884(a0[0], a0[1], gr[1], BrT[1]);
                dmma884(a1[0], a1[1], AsT[1], sm.sgs[buf][(4 + t) * P + g]);
                wk[f][k][0] += a0[0] + a1[0];
                wk[f][k][1] += a0[1] + a1[1];
            }
            if (++q == NS) { q = 0; gphase ^= 1u; }
        }
        // results: w = wk (+ lambda B u), the fused dots sum_l u_l w_l per field; then the u buffers are free again
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            double* wdst = w + f * stride + e * P3 + own;
#pragma unroll
            for (int k = 0; k < P; ++k) {
                const double2 uv = *reinterpret_cast<const double2*>(&sm.u[f][k * P2 + own]);
                double v0 = wk[f][k][0], v1 = wk[f][k][1];
                if (Bm) {
                    const double2 bm = *reinterpret_cast<const double2*>(Bm + e * P3 + own + k * P2);
                    v0 += lambda * bm.x * uv.x;
                    v1 += lambda * bm.y * uv.y;
                }
                *reinterpret_cast<double2*>(wdst + k * P2) = make_double2(v0, v1);
                partial[f] += uv.x * v0 + uv.y * v1;
            }
        }
        __syncwarp();
        if (lane == 0 && n + 1 < nmine) issue_u(n + 1);
    }
    if (dot_out) {
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            double v = partial[f];
            for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) atomicAdd(dot_out + f * dot_stride, v);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int P>
DParam<T, P> make_dparam(const sem_ctx* c) {
    DParam<T, P> d;
    for (int q = 0; q < P * P; ++q) d.D[q] = (T)c->D[q];     // S16: rounded once from double
    return d;
}

Gll1D make_gll(const sem_ctx* c) {
    Gll1D g;
    for (int i = 0; i < 16; ++i) { g.xi[i] = i < c->p ? c->xi[i] : 0.0; g.rho[i] = i < c->p ? c->rho[i] : 0.0; }
    for (int i = 0; i < 256; ++i) g.D[i] = 0.0;              // only xi/rho are used by the Ax kernels
    return g;
}

// Resident CTAs per SM of one kernel instantiation with its dynamic shared memory, cached per device (the opt-in
// attribute is per device as well).  Keyed by the kernel's ADDRESS: two instantiations can share one function-pointer
// type (ax_stream<double,10,..> and ax_pencil<double,10,..>; ax_dmma<3,12> and ax_dmma<5,8>), so a table per type would
// hand the second one the first one's occupancy and never raise its shared-memory limit.
template <typename K>
int resident_blocks(sem_ctx* c, K kern, int threads, size_t smem, int* out) {
    static std::mutex mu;
    static std::map<const void*, std::array<int, SEM_MAX_DEVICES>> tables;
    std::lock_guard<std::mutex> lk(mu);
    const bool cacheable = c->device >= 0 && c->device < SEM_MAX_DEVICES;
    std::array<int, SEM_MAX_DEVICES>* table = nullptr;
    if (cacheable) {
        auto it = tables.find((const void*)kern);
        if (it == tables.end()) it = tables.emplace((const void*)kern, std::array<int, SEM_MAX_DEVICES>{}).first;
        table = &it->second;
    }
    if (!cacheable || !(*table)[c->device]) {
        int nb = 0;
        SEM_CUDA_OK(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        SEM_CUDA_OK(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, threads, smem));
        if (nb < 1) return sem_fail(c, SEM_ECUDA, "Ax kernel does not fit on an SM");
        if (!cacheable) { *out = nb; return SEM_OK; }
        (*table)[c->device] = nb;
    }
    *out = (*table)[c->device];
    return SEM_OK;
}

// u is loaded with the L2 evict-last policy only when a field is small enough to survive in L2 until its next use (config
// 2: the next application, or the next kernel of a PCG iteration, finds it there); a field that streams anyway must not
// crowd out the w values the gather-scatter is about to re-read
inline int u_keep(const sem_ctx* c, size_t bytes_per_node) { return (size_t)c->nL * bytes_per_node <= ((size_t)40 << 20); }

// element range of this launch: everything, or the chunk sem_launch_ax_gs is working on (whole element groups)
struct ElemRange { int64_t e0, ne; };
inline ElemRange elem_range(const sem_ctx* c) { return c->rng_ne > 0 ? ElemRange{c->rng_e0, c->rng_ne} : ElemRange{0, c->E}; }

template <typename T, int P, bool RECOMP>
int launch_simple(sem_ctx* c, const T* u, T* w, T lambda, const int* skip, double* dot) {
    constexpr int EPB = epb_of<P>(), P3 = P * P * P;
    const ElemRange r = elem_range(c);                   // a sub-range of whole element groups, or everything
    const int64_t ngroups = (r.ne + EPB - 1) / EPB;
    const int64_t slab = sizeof(T) == 8 ? c->slab_f64 : c->slab_f32;
    const T* Gs = (sizeof(T) == 8 ? (const T*)c->d_G : (const T*)c->d_G32) + (r.e0 / EPB) * P * EPB * slab;
    const T* Bm = sizeof(T) == 8 ? (const T*)c->d_B : (const T*)c->d_B32;
    const unsigned grid = (unsigned)(ngroups < (int64_t)c->num_sms * 32 ? ngroups : (int64_t)c->num_sms * 32);
    const DParam<T, P> dp = make_dparam<T, P>(c);
    const Gll1D gll = make_gll(c);
    ax_simple<T, P, RECOMP><<<grid, threads_of<P>(), 0, c->stream>>>(
        r.ne, dp, gll, slab, Gs, c->d_vert + r.e0 * 24, (lambda != T(0) && Bm) ? Bm + r.e0 * P3 : nullptr, lambda, u + r.e0 * P3,
        w + r.e0 * P3, skip, dot);
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

template <typename T, int P, int NS, int MINB, bool RG = false>
int launch_stream(sem_ctx* c, const T* u, T* w, T lambda, const int* skip, double* dot) {
    using SM = StreamSmem<T, P, NS, RG>;
    constexpr int EPB = epb_of<P>(), P3 = P * P * P;
    const ElemRange r = elem_range(c);
    const int64_t ngroups = (r.ne + EPB - 1) / EPB;
    const T* Gs = RG ? nullptr
                     : (sizeof(T) == 8 ? (const T*)c->d_G : (const T*)c->d_G32) + (r.e0 / EPB) * P * EPB * SM::SLAB;
    const T* Bm = sizeof(T) == 8 ? (const T*)c->d_B : (const T*)c->d_B32;
    const DParam<T, P> dp = make_dparam<T, P>(c);
    GllP<T, P> gl;
    for (int q = 0; q < P; ++q) { gl.xi[q] = (T)c->xi[q]; gl.rho[q] = (T)c->rho[q]; }
    const size_t smem = sizeof(SM) + 128;
    auto kern = ax_stream<T, P, NS, MINB, RG>;
    int blocks_per_sm = 0;
    if (int rc = resident_blocks(c, kern, threads_of<P>(), smem, &blocks_per_sm)) return rc;
    const int64_t cap = (int64_t)c->num_sms * blocks_per_sm;
    const unsigned grid = (unsigned)(ngroups < cap ? ngroups : cap);
    kern<<<grid, threads_of<P>(), smem, c->stream>>>(r.ne, dp, Gs, (lambda != T(0) && Bm) ? Bm + r.e0 * P3 : (const T*)nullptr,
                                                     lambda, u + r.e0 * P3, w + r.e0 * P3, skip, dot, u_keep(c, sizeof(T)),
                                                     RG ? c->d_vert + r.e0 * 24 : (const double*)nullptr, gl);
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

template <typename T, int P, int NS, int MINB>
int launch_pencil(sem_ctx* c, const T* u, T* w, T lambda, const int* skip, double* dot) {
    using SM = PencilSmem<T, P, NS>;
    constexpr int P3 = P * P * P;
    const ElemRange r = elem_range(c);
    const T* Gs = (sizeof(T) == 8 ? (const T*)c->d_G : (const T*)c->d_G32) + r.e0 * P * SM::SLAB;
    const T* Bm = sizeof(T) == 8 ? (const T*)c->d_B : (const T*)c->d_B32;
    const DParam<T, P> dp = make_dparam<T, P>(c);
    const size_t smem = sizeof(SM) + 128;
    auto kern = ax_pencil<T, P, NS, MINB>;
    int blocks_per_sm = 0;
    if (int rc = resident_blocks(c, kern, threads_of<P>(), smem, &blocks_per_sm)) return rc;
    const int64_t cap = (int64_t)c->num_sms * blocks_per_sm;
    const unsigned grid = (unsigned)(r.ne < cap ? r.ne : cap);
    kern<<<grid, threads_of<P>(), smem, c->stream>>>(r.ne, dp, Gs, lambda != T(0) ? Bm + r.e0 * P3 : (const T*)nullptr,
                                                     lambda, u + r.e0 * P3, w + r.e0 * P3, skip, dot, u_keep(c, sizeof(T)));
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

template <int NS, int MINB, int NU = 2>
int launch_dmma(sem_ctx* c, const double* u, double* w, double lambda, const int* skip, double* dot) {
    using SM = DmmaSmem<NS, NU>;
    const DParam<double, 8> dp = make_dparam<double, 8>(c);
    const size_t smem = sizeof(SM) + 128;
    auto kern = ax_dmma<NS, MINB, NU>;
    int blocks_per_sm = 0;
    if (int rc = resident_blocks(c, kern, 32, smem, &blocks_per_sm)) return rc;
    const ElemRange r = elem_range(c);
    const int64_t cap = (int64_t)c->num_sms * blocks_per_sm;
    const unsigned grid = (unsigned)(r.ne < cap ? r.ne : cap);
    kern<<<grid, 32, smem, c->stream>>>(r.ne, dp, c->d_G + r.e0 * (8 * 6 * 64),
                                        lambda != 0.0 ? c->d_B + r.e0 * 512 : (const double*)nullptr, lambda,
                                        u + r.e0 * 512, w + r.e0 * 512, skip, dot, u_keep(c, 8));
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

template <int MINB, int NU = 2>
int launch_dmma_rg(sem_ctx* c, const double* u, double* w, double lambda, const int* skip, double* dot) {
    using SM = DmmaRgSmem<NU>;
    const DParam<double, 8> dp = make_dparam<double, 8>(c);
    GllP8 gll;
    for (int i = 0; i < 8; ++i) { gll.xi[i] = c->xi[i]; gll.rho[i] = c->rho[i]; }
    const size_t smem = sizeof(SM) + 128;
    auto kern = lambda != 0.0 ? ax_dmma_rg<MINB, NU, true> : ax_dmma_rg<MINB, NU, false>;
    int blocks_per_sm = 0;
    if (int rc = resident_blocks(c, kern, 32, smem, &blocks_per_sm)) return rc;
    const ElemRange r = elem_range(c);
    const int64_t cap = (int64_t)c->num_sms * blocks_per_sm;
    const unsigned grid = (unsigned)(r.ne < cap ? r.ne : cap);
    kern<<<grid, 32, smem, c->stream>>>(r.ne, dp, gll, c->d_vert + r.e0 * 24, lambda, u + r.e0 * 512, w + r.e0 * 512, skip, dot,
                                        u_keep(c, 8));
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

template <int NS, int MINB>
int launch_tf32(sem_ctx* c, const float* u, float* w, float lambda, const int* skip, double* dot) {
    using SM = Tf32Smem<NS>;
    const DParam<float, 8> dp = make_dparam<float, 8>(c);
    const size_t smem = sizeof(SM) + 128;
    auto kern = ax_tf32<NS, MINB>;
    int blocks_per_sm = 0;
    if (int rc = resident_blocks(c, kern, 32, smem, &blocks_per_sm)) return rc;
    const ElemRange r = elem_range(c);
    const int64_t cap = (int64_t)c->num_sms * blocks_per_sm;
    const unsigned grid = (unsigned)(r.ne < cap ? r.ne : cap);
    kern<<<grid, 32, smem, c->stream>>>(r.ne, dp, c->d_G32 + r.e0 * (8 * 6 * 64),
                                        lambda != 0.f ? c->d_B32 + r.e0 * 512 : (const float*)nullptr, lambda,
                                        u + r.e0 * 512, w + r.e0 * 512, skip, dot, u_keep(c, 4));
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

template <int NF>
int launch_dmma_many(sem_ctx* c, const double* u, double* w, int64_t stride, double lambda, const int* skip, double* dot,
                     int64_t dot_stride) {
    constexpr int NS = 3, MINB = 8;
    using SM = DmmaManySmem<NF, NS>;
    const DParam<double, 8> dp = make_dparam<double, 8>(c);
    const size_t smem = sizeof(SM) + 128;
    auto kern = ax_dmma_many<NF, NS, MINB>;
    int blocks_per_sm = 0;
    if (int rc = resident_blocks(c, kern, 32, smem, &blocks_per_sm)) return rc;
    const int64_t cap = (int64_t)c->num_sms * blocks_per_sm;
    const unsigned grid = (unsigned)(c->E < cap ? c->E : cap);
    kern<<<grid, 32, smem, c->stream>>>(c->E, dp, c->d_G, lambda != 0.0 ? c->d_B : (const double*)nullptr, lambda, u, w,
                                        stride, skip, dot, dot_stride, u_keep(c, 8 * NF));
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

// stage depth / residency per (T, P): sized so that ~7-8 CTAs fit in 227 KB and > 64 KB are in flight per SM
template <typename T, int P> struct StreamCfg { static constexpr int NS = 4, MINB = 1; };
template <> struct StreamCfg<double, 8> { static constexpr int NS = 5, MINB = 8; };
template <> struct StreamCfg<float, 8> { static constexpr int NS = 8, MINB = 8; };
template <> struct StreamCfg<double, 2> { static constexpr int NS = 2, MINB = 8; };
template <> struct StreamCfg<float, 2> { static constexpr int NS = 2, MINB = 8; };
template <> struct StreamCfg<double, 4> { static constexpr int NS = 4, MINB = 8; };
template <> struct StreamCfg<float, 4> { static constexpr int NS = 4, MINB = 8; };
template <> struct StreamCfg<double, 6> { static constexpr int NS = 5, MINB = 5; };
template <> struct StreamCfg<float, 6> { static constexpr int NS = 6, MINB = 6; };
template <> struct StreamCfg<double, 10> { static constexpr int NS = 4, MINB = 3; };
template <> struct StreamCfg<float, 10> { static constexpr int NS = 6, MINB = 4; };

template <int P> constexpr bool stream_ok() { return P <= 12; }
// resident CTAs the recomputed-G instantiation is compiled for (15 more live values per thread than the stored-G one)
// (FP64-pipe bound, little shared memory: registers first, occupancy second)
template <typename T, int P> struct StreamCfgRG {
    static constexpr int WANT = sizeof(T) == 8 ? (P >= 9 ? 255 : P >= 7 ? 208 : 168) : (P >= 11 ? 192 : 128);   // registers per thread
    static constexpr int FIT = 65536 / (threads_of<P>() * WANT);
    static constexpr int MINB = FIT < 1 ? 1 : (FIT > 8 ? 8 : FIT);
};
template <> struct StreamCfg<double, 9> { static constexpr int NS = 4, MINB = 4; };
template <> struct StreamCfg<float, 9> { static constexpr int NS = 6, MINB = 5; };
template <> struct StreamCfg<double, 7> { static constexpr int NS = 4, MINB = 4; };
template <> struct StreamCfg<float, 7> { static constexpr int NS = 5, MINB = 6; };
template <> struct StreamCfg<double, 5> { static constexpr int NS = 4, MINB = 6; };
template <> struct StreamCfg<float, 5> { static constexpr int NS = 4, MINB = 8; };
template <> struct StreamCfg<double, 3> { static constexpr int NS = 3, MINB = 8; };
template <> struct StreamCfg<float, 3> { static constexpr int NS = 3, MINB = 8; };

template <typename T, int P>
int dispatch_p(sem_ctx* c, const void* u, void* w, double lambda, const int* skip, double* dot) {
    const T* uu = (const T*)u;
    T* ww = (T*)w;
    const bool aligned = ((uintptr_t)u % 16) == 0;
    if (c->gmode == SEM_G_RECOMPUTE) {
        if constexpr (P == 8 && sizeof(T) == 8) {      // a9 on the tensor cores, no G traffic; variant 1 keeps ax_simple
            if (aligned && c->ax_variant != 1 && c->ax_variant != 2)
                return launch_dmma_rg<8>(c, (const double*)u, (double*)w, lambda, skip, dot);
        }
        if constexpr (stream_ok<P>()) {                // every other p <= 12 (and variant 2): the streaming kernel, no G ring
            if (aligned && c->ax_variant != 1)
                return launch_stream<T, P, 1, StreamCfgRG<T, P>::MINB, true>(c, uu, ww, (T)lambda, skip, dot);
        }
        return launch_simple<T, P, true>(c, uu, ww, (T)lambda, skip, dot);
    }
    // variant 0: the default kernel per (T, p): p = 8 runs on the tensor cores (FP64: DMMA, FP32: TF32 x 3);
    // 1: ax_simple; 2: ax_stream (scalar contractions); 3: FP64 p = 8: the DMMA kernel with 5 stages / 8 warps per SM
    if constexpr (P == 8 && sizeof(T) == 8) {
        if (aligned && c->ax_variant == 0) return launch_dmma<3, 12>(c, (const double*)u, (double*)w, lambda, skip, dot);
        if (aligned && c->ax_variant == 3) return launch_dmma<5, 8>(c, (const double*)u, (double*)w, lambda, skip, dot);
    }
    if constexpr (P == 8 && sizeof(T) == 4) {          // FP32 p = 8: the TF32 x 3 tensor-core kernel
        if (aligned && c->ax_variant == 0) return launch_tf32<3, 12>(c, (const float*)u, (float*)w, (float)lambda, skip, dot);
    }
    // the pencil kernel (variant 4, p = 8 ... 12): the default only where it measured faster than ax_stream
    if constexpr (P >= 8 && P <= 12) {
        constexpr bool WINS = (sizeof(T) == 4 && P == 9) || (sizeof(T) == 8 && P == 12);
        if (aligned && (c->ax_variant == 4 || (WINS && c->ax_variant == 0)))
            return launch_pencil<T, P, 4, (P == 8 ? 8 : sizeof(T) == 8 ? 4 : 5)>(c, uu, ww, (T)lambda, skip, dot);
    }
    if constexpr (stream_ok<P>()) {
        if (c->ax_variant != 1 && aligned)
            return launch_stream<T, P, StreamCfg<T, P>::NS, StreamCfg<T, P>::MINB>(c, uu, ww, (T)lambda, skip, dot);
    }
    return launch_simple<T, P, false>(c, uu, ww, (T)lambda, skip, dot);
}

template <typename T>
int dispatch(sem_ctx* c, const void* u, void* w, double lambda, const int* skip, double* dot) {
    switch (c->p) {
#define SEM_CASE(PP) case PP: return dispatch_p<T, PP>(c, u, w, lambda, skip, dot);
        SEM_CASE(2) SEM_CASE(3) SEM_CASE(4) SEM_CASE(5) SEM_CASE(6) SEM_CASE(7) SEM_CASE(8) SEM_CASE(9)
        SEM_CASE(10) SEM_CASE(11) SEM_CASE(12) SEM_CASE(13) SEM_CASE(14) SEM_CASE(15) SEM_CASE(16)
#undef SEM_CASE
    }
    return sem_fail(c, SEM_EINVAL, "unsupported p = %d", c->p);
}

}  // namespace

// dot_out != nullptr: also accumulate sum_l u_l w_l (the un-assembled local dot, O8) into *dot_out (device, FP64).
// skip_flag != nullptr: the kernel returns at once if *skip_flag != 0 (device; used by the PCG loop after convergence).
int sem_launch_ax(sem_ctx* c, const void* u, void* w, sem_prec prec, double lambda, double* dot_out,
                  const int* skip_flag) {
    if (prec == SEM_F64) return dispatch<double>(c, u, w, lambda, skip_flag, dot_out);
    return dispatch<float>(c, u, w, lambda, skip_flag, dot_out);
}

// a3-a7: the local operator followed by the gather-scatter kernel (sem_gs.cu), which also applies the Dirichlet mask.
// (Single-launch variants -- an owner-computes epilogue, concurrently running gather-scatter workers, a gather-scatter
// tail phase of the operator kernel -- were built and measured slower than the two launches.)
int sem_launch_ax_gs(sem_ctx* c, const void* u, void* w, sem_prec prec, double lambda, double* dot_out,
                     const int* skip_flag) {
    int rc;
    const int nch = (int)c->chunk_e0.size() - 1;
    if (nch < 2) {
        if ((rc = sem_launch_ax(c, u, w, prec, lambda, dot_out, skip_flag))) return rc;
        return sem_launch_gs(c, w, prec, true, skip_flag);
    }
    // The field does not fit in L2 (the gather-scatter then runs at 2x its bytes in DRAM sectors):
    // operator and gather-scatter alternate chunk by chunk.  The records are sorted by the element group of a node's LAST
    // copy, so the records of chunk q only touch values written by chunks <= q, a few tens of MB ago: still in L2 for any
    // element order with locality (every box mesh in lexicographic order; not config 5's scrambled order).
    return sem_launch_ax_gs_chunks(c, u, w, prec, lambda, dot_out, skip_flag, 0, nch);
}

// chunks [q0, q1) of the chunked operator + gather-scatter (the sharded apply starts its exchange between two ranges)
int sem_launch_ax_gs_chunks(sem_ctx* c, const void* u, void* w, sem_prec prec, double lambda, double* dot_out,
                            const int* skip_flag, int q0, int q1) {
    int rc;
    for (int q = q0; q < q1; ++q) {
        c->rng_e0 = c->chunk_e0[q];
        c->rng_ne = c->chunk_e0[q + 1] - c->chunk_e0[q];
        rc = c->rng_ne > 0 ? sem_launch_ax(c, u, w, prec, lambda, dot_out, skip_flag) : SEM_OK;
        c->rng_ne = 0;
        if (rc) return rc;
        if ((rc = sem_launch_gs_range(c, w, prec, true, skip_flag, q))) return rc;
    }
    return SEM_OK;
}

// NEXT-4: the operator on nf fields (u + f * stride -> w + f * stride).  FP64 p = 8 with stored G and 16-byte aligned
// fields: groups of 3 (or 2) fields share one pass over G (ax_dmma_many); everything else: field by field.
// dot_out + f * dot_stride receives sum_l u_l w_l of field f (nullptr: none).
int sem_launch_ax_many(sem_ctx* c, const void* u, void* w, int nf, int64_t stride, sem_prec prec, double lambda,
                       double* dot_out, int64_t dot_stride, const int* skip_flag) {
    const size_t vs = prec == SEM_F64 ? 8 : 4;
    const bool fused = prec == SEM_F64 && c->p == 8 && c->gmode == SEM_G_STORED && c->ax_variant == 0 &&
                       ((uintptr_t)u % 16) == 0 && ((uintptr_t)w % 16) == 0 && (stride % 2) == 0;
    int f = 0, rc;
    while (f < nf) {
        const int left = nf - f;
        const int take = !fused ? 1 : (left >= 3 && left != 4 ? 3 : (left >= 2 ? 2 : 1));
        const char* uf = (const char*)u + (size_t)f * (size_t)stride * vs;
        char* wf = (char*)w + (size_t)f * (size_t)stride * vs;
        double* df = dot_out ? dot_out + f * dot_stride : nullptr;
        if (take == 3) rc = launch_dmma_many<3>(c, (const double*)uf, (double*)wf, stride, lambda, skip_flag, df, dot_stride);
        else if (take == 2) rc = launch_dmma_many<2>(c, (const double*)uf, (double*)wf, stride, lambda, skip_flag, df, dot_stride);
        else rc = sem_launch_ax(c, uf, wf, prec, lambda, df, skip_flag);
        if (rc) return rc;
        f += take;
    }
    return SEM_OK;
}
