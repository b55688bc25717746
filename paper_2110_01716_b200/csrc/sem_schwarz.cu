// sem_schwarz.cu — NEXT-2b: the overlapping additive Schwarz smoother around the fast-diagonalisation
// local solve of sem_fdm.cu.  P:103 "The Schwarz smoothers are implemented by solving local Poisson problems on domains
// extended into adjacent elements by one layer.  Thus, for an 8 x 8 x 8 brick (N = 7), one solves a 10 x 10 x 10 local
// problem, A~ u~ = b~, using fast diagonalization", Eq. (3); "We exchange face data only to get the domain
// extensions -- meaning 6 exchanges per element instead of 26 ... a restricted additive Schwarz (RAS) variant, that does
// not require communication after the local solve"; P:109 FP32; Table 2 `gs_ext`, `fdm`, `fdm_apply`.
// The paper cites Lottes & Fischer (2005) for the construction and prints none of it: what is built here is reading S29
// of DESIGN.md (restated at sem_schwarz_setup in include/sem.h):
//   z = M W^1/2 QQ^T sum_e R_e^T A~_e^-1 R_e (W^1/2 r),  A~_e = Bz x By x Ax + Bz x Ay x Bx + Az x By x Bx  (m = N + 3)
// Three kernels per application, all element-local reads of a continuous field (the "exchange" is a gather through
// the face links resolved at setup, so there is no pack/unpack and no atomics):
//   k_schwarz_ext      b~_e: the element's own residual in the block's interior, the face neighbour's one-layer-in
//                      values in its 6 face layers (`gs_ext`), zero on the block's edges and corners;
//   sem_fdm_apply      Eq. (3) in place on the blocks;
//   k_schwarz_combine  z_L = W (own part of u~_e + the neighbours' ghost-layer values that land on this element's
//                      one-layer-in nodes); then the ordinary gather-scatter with the Dirichlet mask sums the copies.
#include <math.h>

#include <vector>

#include "sem_internal.h"

struct sem_schwarz_data {
    int m = 0;
    int4* d_link = nullptr;        // [E][6]  (nbr element or -1, base, sa, sb): neighbour's local index of the node that
                                   //         matches my face node (fa, fb) is base + fa * sa + fb * sb
    int32_t* d_nrm = nullptr;      // [E][6]  neighbour's face: axis (0,1,2 = i,j,k) | side << 2 (0: index 0, 1: index N)
    std::vector<double> hA, hB;    // host copies of the 1-D operator pairs [E][3][m][m] (parity accessor)
    std::vector<int32_t> hnbr;     // [E][6]
    double *d_S64 = nullptr, *d_iL64 = nullptr;
    float *d_S32 = nullptr, *d_iL32 = nullptr;
    // weights in local layout, [ASM, RAS]: ASM holds sqrt(W) (applied to r before the extension and to the combined
    // result: S stays symmetric), RAS holds W = 1 / multiplicity (applied to the result only)
    double* d_W64[2] = {nullptr, nullptr};
    float* d_W32[2] = {nullptr, nullptr};
    void* d_ext = nullptr;         // [E][m^3] work blocks (sized for doubles)
};

void sem_schwarz_free(sem_ctx* c) {
    sem_schwarz_data* s = c->sw;
    if (!s) return;
    void* ptrs[] = {s->d_link, s->d_nrm, s->d_S64, s->d_iL64, s->d_S32, s->d_iL32, s->d_W64[0], s->d_W64[1], s->d_W32[0],
                    s->d_W32[1], s->d_ext};
    for (void* p : ptrs) cudaFree(p);
    cudaGetLastError();
    delete s;
    c->sw = nullptr;
}

namespace {

// face f = 2 * axis + side.  Face coordinates (fa, fb) of a face of axis 0 (i fixed): (j, k); axis 1: (i, k); axis 2: (i, j).
__host__ __device__ inline int face_node(int p, int axis, int side, int fa, int fb) {
    const int fix = side ? p - 1 : 0;
    const int i = axis == 0 ? fix : fa;
    const int j = axis == 0 ? fa : (axis == 1 ? fix : fb);
    const int k = axis == 2 ? fix : fb;
    return (k * p + j) * p + i;
}

// one-layer-in node of the face neighbour behind my face node (fa, fb), and the block position of the neighbour's ghost
// node that lies on my one-layer-in node (fa, fb) of that face
__device__ __forceinline__ int nbr_one_in(int p, const int4 lk, int nf, int fa, int fb) {
    const int na = nf & 3, ns = nf >> 2;
    const int stride = na == 0 ? 1 : (na == 1 ? p : p * p);
    return lk.y + fa * lk.z + fb * lk.w + (ns ? -stride : stride);
}
__device__ __forceinline__ int nbr_ghost_pos(int p, const int4 lk, int nf, int fa, int fb) {
    const int m = p + 2, na = nf & 3, ns = nf >> 2;
    const int ln = lk.y + fa * lk.z + fb * lk.w;                               // neighbour's face node behind mine
    int ci = ln % p + 1, cj = (ln / p) % p + 1, ck = ln / (p * p) + 1;          // block coordinates
    if (na == 0) ci += ns ? 1 : -1;                                             // one step OUT of the neighbour
    else if (na == 1) cj += ns ? 1 : -1;
    else ck += ns ? 1 : -1;
    return (ck * m + cj) * m + ci;
}

// b~ (`gs_ext`): one CTA per element.  Three index ranges instead of a test per block position: the p^3 own nodes, the
// 6 p^2 face-layer entries (gathered from the neighbours), the 12 p + 8 edge and corner positions (zero).
// PC: p at compile time for the orders of the paper's level schedules (0: run-time p).
template <typename T, int PC>
__global__ void __launch_bounds__(256) k_schwarz_ext(int64_t E, int p_rt, const int4* __restrict__ link_g,
                                                     const int32_t* __restrict__ nrm_g, const T* __restrict__ r,
                                                     const T* __restrict__ pre, T* __restrict__ ext) {
    const int p = PC ? PC : p_rt;
    const int m = p + 2, m2 = m * m, m3 = m2 * m, p2 = p * p, p3 = p2 * p;
    __shared__ int4 link[6];
    __shared__ int32_t nrm[6];
    for (int64_t e = blockIdx.x; e < E; e += gridDim.x) {
        __syncthreads();
        if (threadIdx.x < 6) { link[threadIdx.x] = link_g[e * 6 + threadIdx.x]; nrm[threadIdx.x] = nrm_g[e * 6 + threadIdx.x]; }
        __syncthreads();
        T* xe = ext + e * m3;
        for (int l = threadIdx.x; l < p3; l += blockDim.x) {                    // own nodes
            const int i = l % p, j = (l / p) % p, k = l / p2;
            const T v = pre ? pre[e * p3 + l] * r[e * p3 + l] : r[e * p3 + l];
            xe[(k + 1) * m2 + (j + 1) * m + (i + 1)] = v;
        }
        for (int t = threadIdx.x; t < 6 * p2; t += blockDim.x) {                // face layers
            const int f = t / p2, fa = (t % p2) % p, fb = (t % p2) / p;
            const int axis = f >> 1, g = (f & 1) ? m - 1 : 0;
            const int a = axis == 0 ? g : fa + 1, b = axis == 0 ? fa + 1 : (axis == 1 ? g : fb + 1),
                      c = axis == 2 ? g : fb + 1;
            const int4 lk = link[f];
            T v = T(0);
            if (lk.x >= 0) {
                const int64_t src = (int64_t)lk.x * p3 + nbr_one_in(p, lk, nrm[f], fa, fb);
                v = pre ? pre[src] * r[src] : r[src];
            }
            xe[c * m2 + b * m + a] = v;
        }
        for (int t = threadIdx.x; t < 12 * p + 8; t += blockDim.x) {            // edges and corners of the block: no node
            int a, b, c;
            if (t < 12 * p) {
                const int ed = t / p, q = t % p + 1, ax = ed >> 2, s0 = (ed & 1) ? m - 1 : 0, s1 = (ed & 2) ? m - 1 : 0;
                a = ax == 0 ? q : s0;
                b = ax == 1 ? q : (ax == 0 ? s0 : s1);
                c = ax == 2 ? q : s1;
            } else {
                const int cn = t - 12 * p;
                a = (cn & 1) ? m - 1 : 0; b = (cn & 2) ? m - 1 : 0; c = (cn & 4) ? m - 1 : 0;
            }
            xe[c * m2 + b * m + a] = T(0);
        }
    }
}

// z_L = W (own part of u~ + ghost layers of the face neighbours): the own part goes to shared memory, the 6 p^2 ghost
// values are loaded together, and are added face by face (a node of two one-layer-in planes receives its contributions
// in a fixed order: results are bit-repeatable)
template <typename T, bool RESTRICTED, int PC>
__global__ void __launch_bounds__(256) k_schwarz_combine(int64_t E, int p_rt, const int4* __restrict__ link_g,
                                                         const int32_t* __restrict__ nrm_g, const T* __restrict__ ext,
                                                         const T* __restrict__ W, T* __restrict__ z) {
    const int p = PC ? PC : p_rt;
    const int m = p + 2, m2 = m * m, m3 = m2 * m, p2 = p * p, p3 = p2 * p, N = p - 1;
    __shared__ int4 link[6];
    __shared__ int32_t nrm[6];
    extern __shared__ __align__(16) unsigned char zs_raw[];
    T* zs = reinterpret_cast<T*>(zs_raw);                                        // [p^3]
    for (int64_t e = blockIdx.x; e < E; e += gridDim.x) {
        __syncthreads();
        if (threadIdx.x < 6) { link[threadIdx.x] = link_g[e * 6 + threadIdx.x]; nrm[threadIdx.x] = nrm_g[e * 6 + threadIdx.x]; }
        __syncthreads();
        const T* xe = ext + e * m3;
        if (RESTRICTED) {
            for (int l = threadIdx.x; l < p3; l += blockDim.x) {
                const int i = l % p, j = (l / p) % p, k = l / p2;
                const T v = xe[(k + 1) * m2 + (j + 1) * m + (i + 1)];
                z[e * p3 + l] = W ? W[e * p3 + l] * v : v;
            }
            continue;
        }
        // ghost values of the neighbours, two entries per thread at most (6 p^2 <= 2 x 256 up to p = 9; more: loop)
        constexpr int MAXV = 6;
        T gv[MAXV];
        int nv = 0;
        for (int t = threadIdx.x; t < 6 * p2 && nv < MAXV; t += blockDim.x, ++nv) {
            const int f = t / p2, fa = (t % p2) % p, fb = (t % p2) / p;
            const int4 lk = link[f];
            gv[nv] = lk.x >= 0 ? ext[(int64_t)lk.x * m3 + nbr_ghost_pos(p, lk, nrm[f], fa, fb)] : T(0);
        }
        for (int l = threadIdx.x; l < p3; l += blockDim.x) {
            const int i = l % p, j = (l / p) % p, k = l / p2;
            zs[l] = xe[(k + 1) * m2 + (j + 1) * m + (i + 1)];
        }
        __syncthreads();
        for (int f = 0; f < 6; ++f) {
            nv = 0;
            for (int t = threadIdx.x; t < 6 * p2 && nv < MAXV; t += blockDim.x, ++nv) {
                if (t / p2 != f) continue;
                const int fa = (t % p2) % p, fb = (t % p2) / p, axis = f >> 1, q = (f & 1) ? N - 1 : 1;
                const int i = axis == 0 ? q : fa, j = axis == 0 ? fa : (axis == 1 ? q : fb), k = axis == 2 ? q : fb;
                zs[(k * p + j) * p + i] += gv[nv];
            }
            __syncthreads();
        }
        for (int l = threadIdx.x; l < p3; l += blockDim.x) z[e * p3 + l] = W ? W[e * p3 + l] * zs[l] : zs[l];
    }
}

template <typename T>
__global__ void __launch_bounds__(256) k_fill(int64_t n, T v, T* __restrict__ x) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) x[l] = v;
}
// W = 1 / count (count >= 1 at every node: its own position), or its square root; both precisions from the FP64 count
__global__ void __launch_bounds__(256) k_inv_w(int64_t n, const double* __restrict__ cnt, bool root,
                                               double* __restrict__ w64, float* __restrict__ w32) {
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const double w = root ? 1.0 / sqrt(cnt[l]) : 1.0 / cnt[l];
        w64[l] = w;
        w32[l] = (float)w;
    }
}

// p = 8, 6, 4 (N = 7, 5, 3: the upper levels of the 7-3-1 and 8-5-1 / 8-6-4-1 schedules run one order apart) and 9, 7, 5
// are compiled with p fixed; any other order runs the generic instantiation
template <typename T>
void launch_ext(sem_ctx* c, unsigned grid, const T* r, const T* pre, T* ext) {
    sem_schwarz_data* s = c->sw;
#define SEM_SW_EXT(PP) k_schwarz_ext<T, PP><<<grid, 256, 0, c->stream>>>(c->E, c->p, s->d_link, s->d_nrm, r, pre, ext)
    switch (c->p) {
        case 4: SEM_SW_EXT(4); break;  case 5: SEM_SW_EXT(5); break;  case 6: SEM_SW_EXT(6); break;
        case 7: SEM_SW_EXT(7); break;  case 8: SEM_SW_EXT(8); break;  case 9: SEM_SW_EXT(9); break;
        default: SEM_SW_EXT(0);
    }
#undef SEM_SW_EXT
}
template <typename T>
void launch_combine(sem_ctx* c, unsigned grid, bool restricted, const T* ext, const T* W, T* z) {
    sem_schwarz_data* s = c->sw;
#define SEM_SW_CMB(PP)                                                                                            \
    do {                                                                                                          \
        const size_t sm = sizeof(T) * c->p3;                                                                      \
        if (restricted) k_schwarz_combine<T, true, PP><<<grid, 256, sm, c->stream>>>(c->E, c->p, s->d_link, s->d_nrm, ext, W, z); \
        else k_schwarz_combine<T, false, PP><<<grid, 256, sm, c->stream>>>(c->E, c->p, s->d_link, s->d_nrm, ext, W, z);          \
    } while (0)
    switch (c->p) {
        case 4: SEM_SW_CMB(4); break;  case 5: SEM_SW_CMB(5); break;  case 6: SEM_SW_CMB(6); break;
        case 7: SEM_SW_CMB(7); break;  case 8: SEM_SW_CMB(8); break;  case 9: SEM_SW_CMB(9); break;
        default: SEM_SW_CMB(0);
    }
#undef SEM_SW_CMB
}

template <typename T>
int apply(sem_ctx* c, const T* r, T* z, int kind) {
    sem_schwarz_data* s = c->sw;
    const sem_prec prec = sizeof(T) == 8 ? SEM_F64 : SEM_F32;
    const T* S = sizeof(T) == 8 ? (const T*)s->d_S64 : (const T*)s->d_S32;
    const T* iL = sizeof(T) == 8 ? (const T*)s->d_iL64 : (const T*)s->d_iL32;
    const T* W = sizeof(T) == 8 ? (const T*)s->d_W64[kind] : (const T*)s->d_W32[kind];
    T* ext = (T*)s->d_ext;
    const unsigned grid = (unsigned)c->E;
    if (kind == SEM_SCHWARZ_RAS && r != z) {
        // restricted variant: one kernel (gather from r into the shared-memory block, Eq. (3), weighted own part to z)
        // and the gather-scatter; in place (r == z) an element would read neighbour values already overwritten
        int rc1 = sem_launch_fdm_schwarz(c, s->m, S, iL, r, s->d_link, s->d_nrm, W, z, prec);
        if (rc1) return rc1;
        return sem_launch_gs(c, z, prec, /*apply_mask=*/true);
    }
    launch_ext<T>(c, grid, r, kind == SEM_SCHWARZ_ASM ? W : (const T*)nullptr, ext);
    int rc = sem_fdm_apply(c, s->m, S, iL, ext, ext, prec);
    if (rc) return rc;
    launch_combine<T>(c, grid, kind == SEM_SCHWARZ_RAS, ext, W, z);
    SEM_CUDA_OK(c, cudaGetLastError());
    return sem_launch_gs(c, z, prec, /*apply_mask=*/true);
}

}  // namespace

int sem_launch_schwarz(sem_ctx* c, const void* r, void* z, sem_prec prec, int kind) {
    if (prec == SEM_F64) return apply<double>(c, (const double*)r, (double*)z, kind);
    return apply<float>(c, (const float*)r, (float*)z, kind);
}

extern "C" int sem_schwarz_setup(sem_ctx* c) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (!c->geom_done) return sem_fail(c, SEM_ESTATE, "sem_schwarz_setup before sem_geom");
    if (c->N < 2) return sem_fail(c, SEM_EINVAL, "sem_schwarz_setup: needs N >= 2 (a face must have an interior node)");
    if (c->sw) return SEM_OK;
    const int p = c->p, N = c->N, m = p + 2;
    const int64_t E = c->E, p3 = c->p3, m2 = (int64_t)m * m, m3 = m2 * m;
    cudaStream_t st = c->stream;
    // ---- host copies of what the link search needs: canonical maps, unique-node mask, vertices ----
    std::vector<int32_t> l2u(c->nL), seg_idx(c->nL);
    std::vector<int64_t> seg_off(c->U + 1);
    std::vector<uint8_t> mask_u(c->has_mask ? c->U : 0);
    std::vector<double> vert(E * 24);
    SEM_CUDA_OK(c, cudaMemcpyAsync(l2u.data(), c->d_l2u, c->nL * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaMemcpyAsync(seg_idx.data(), c->d_seg_idx, c->nL * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaMemcpyAsync(seg_off.data(), c->d_seg_off, (c->U + 1) * sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    if (c->has_mask) SEM_CUDA_OK(c, cudaMemcpyAsync(mask_u.data(), c->d_mask_u, c->U, cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaMemcpyAsync(vert.data(), c->d_vert, E * 24 * sizeof(double), cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    // ---- element lengths: mean of the 4 edges in each local direction (S29) ----
    std::vector<double> L(E * 3);
    for (int64_t e = 0; e < E; ++e)
        for (int d = 0; d < 3; ++d) {
            double sum = 0.0;
            for (int v = 0; v < 8; ++v) {
                if ((v >> d) & 1) continue;
                const double* a = &vert[(e * 8 + v) * 3];
                const double* b = &vert[(e * 8 + v + (1 << d)) * 3];
                sum += sqrt((b[0] - a[0]) * (b[0] - a[0]) + (b[1] - a[1]) * (b[1] - a[1]) + (b[2] - a[2]) * (b[2] - a[2]));
            }
            L[e * 3 + d] = 0.25 * sum;
        }
    // ---- face links ----
    sem_schwarz_data* s = new sem_schwarz_data();
    s->m = m;
    s->hnbr.assign(E * 6, -1);
    std::vector<int4> link(E * 6, make_int4(-1, 0, 0, 0));
    std::vector<int32_t> nrm(E * 6, 0);
    std::vector<uint8_t> dirf(E * 6, 0);
    std::vector<double> Lnb(E * 6, -1.0);
    auto copy_in = [&](int32_t g, int64_t n) -> int32_t {          // local index (within element n) of unique node g
        for (int64_t q = seg_off[g]; q < seg_off[g + 1]; ++q)
            if (seg_idx[q] / p3 == n) return (int32_t)(seg_idx[q] - n * p3);
        return -1;
    };
    const int c0 = p / 2;
    for (int64_t e = 0; e < E; ++e)
        for (int f = 0; f < 6; ++f) {
            const int axis = f / 2, side = f % 2;
            const int32_t gc = l2u[e * p3 + face_node(p, axis, side, c0, c0)];
            int64_t n = -1;
            const int64_t cnt = seg_off[gc + 1] - seg_off[gc];
            if (cnt == 2) {
                const int64_t e0 = seg_idx[seg_off[gc]] / p3, e1 = seg_idx[seg_off[gc] + 1] / p3;
                n = e0 == e ? e1 : e0;
                if (n == e) n = -1;                                  // a face glued to itself: treat as a boundary
            }
            if (n < 0) { dirf[e * 6 + f] = c->has_mask && mask_u[gc]; continue; }
            const int32_t l00 = copy_in(l2u[e * p3 + face_node(p, axis, side, 0, 0)], n);
            const int32_t l10 = copy_in(l2u[e * p3 + face_node(p, axis, side, 1, 0)], n);
            const int32_t l01 = copy_in(l2u[e * p3 + face_node(p, axis, side, 0, 1)], n);
            if (l00 < 0 || l10 < 0 || l01 < 0) { delete s; return sem_fail(c, SEM_EMESH, "sem_schwarz_setup: non-conforming face"); }
            int na = -1, ns = 0;
            for (int a = 0, str = 1; a < 3; ++a, str *= p) {
                const int q0 = (l00 / str) % p, q1 = (l10 / str) % p, q2 = (l01 / str) % p;
                if (q0 == q1 && q0 == q2 && (q0 == 0 || q0 == N)) { na = a; ns = q0 == N; }
            }
            if (na < 0) { delete s; return sem_fail(c, SEM_EMESH, "sem_schwarz_setup: cannot orient a shared face"); }
            s->hnbr[e * 6 + f] = (int32_t)n;
            link[e * 6 + f] = make_int4((int)n, l00, l10 - l00, l01 - l00);
            nrm[e * 6 + f] = na | (ns << 2);
            Lnb[e * 6 + f] = L[n * 3 + na];
        }
    // ---- 1-D operator pairs on the extended lines (S29) and their eigen-decompositions (sem_fdm_setup) ----
    std::vector<double> Kh((size_t)p * p, 0.0);                      // reference stiffness D^T diag(rho) D
    for (int a = 0; a < p; ++a)
        for (int b = 0; b < p; ++b) {
            double v = 0.0;
            for (int q = 0; q < p; ++q) v += c->D[q * p + a] * c->rho[q] * c->D[q * p + b];
            Kh[a * p + b] = v;
        }
    s->hA.assign(E * 3 * m2, 0.0);
    s->hB.assign(E * 3 * m2, 0.0);
    for (int64_t e = 0; e < E; ++e)
        for (int d = 0; d < 3; ++d) {
            double* A = &s->hA[(e * 3 + d) * m2];
            double* B = &s->hB[(e * 3 + d) * m2];
            const double Lm = L[e * 3 + d], Ll = Lnb[e * 6 + 2 * d], Lr = Lnb[e * 6 + 2 * d + 1];
            for (int a = 0; a < p; ++a) {
                for (int b = 0; b < p; ++b) A[(a + 1) * m + (b + 1)] += 2.0 / Lm * Kh[a * p + b];
                B[(a + 1) * m + (a + 1)] += 0.5 * Lm * c->rho[a];
            }
            if (Ll > 0.0) {
                for (int a = 0; a < 2; ++a) {
                    for (int b = 0; b < 2; ++b) A[a * m + b] += 2.0 / Ll * Kh[(N - 1 + a) * p + (N - 1 + b)];
                    B[a * m + a] += 0.5 * Ll * c->rho[N - 1 + a];
                }
            } else {
                A[0] = 1.0; B[0] = 1.0;
                if (dirf[e * 6 + 2 * d]) {
                    for (int q = 0; q < m; ++q) A[1 * m + q] = A[q * m + 1] = 0.0;
                    A[1 * m + 1] = 1.0; B[1 * m + 1] = 1.0;
                }
            }
            if (Lr > 0.0) {
                for (int a = 0; a < 2; ++a) {
                    for (int b = 0; b < 2; ++b) A[(m - 2 + a) * m + (m - 2 + b)] += 2.0 / Lr * Kh[a * p + b];
                    B[(m - 2 + a) * m + (m - 2 + a)] += 0.5 * Lr * c->rho[a];
                }
            } else {
                A[(m - 1) * m + (m - 1)] = 1.0; B[(m - 1) * m + (m - 1)] = 1.0;
                if (dirf[e * 6 + 2 * d + 1]) {
                    for (int q = 0; q < m; ++q) A[(m - 2) * m + q] = A[q * m + (m - 2)] = 0.0;
                    A[(m - 2) * m + (m - 2)] = 1.0; B[(m - 2) * m + (m - 2)] = 1.0;
                }
            }
        }
    std::vector<double> S(E * 3 * m2), iL(E * m3);
    int rc = sem_fdm_setup(E, m, s->hA.data(), s->hB.data(), S.data(), iL.data());
    if (rc) { delete s; return sem_fail(c, rc, "sem_schwarz_setup: eigen-decomposition of a 1-D operator pair failed"); }
    for (int64_t e = 0; e < E; ++e) {                                // an all-Neumann block has one zero eigenvalue sum
        double mn = iL[e * m3];
        for (int64_t q = 1; q < m3; ++q) mn = iL[e * m3 + q] < mn ? iL[e * m3 + q] : mn;      // 1 / largest sum
        for (int64_t q = 0; q < m3; ++q)
            if (!(iL[e * m3 + q] > 0.0) || iL[e * m3 + q] > 1e12 * mn) iL[e * m3 + q] = 0.0;
    }
    std::vector<float> S32(S.size()), iL32(iL.size());
    for (size_t q = 0; q < S.size(); ++q) S32[q] = (float)S[q];                              // S16: rounded once
    for (size_t q = 0; q < iL.size(); ++q) iL32[q] = (float)iL[q];
    c->sw = s;
    auto up = [&](void** d, const void* h, size_t bytes) -> cudaError_t {
        cudaError_t e = cudaMalloc(d, bytes ? bytes : 1);
        if (e == cudaSuccess) e = cudaMemcpyAsync(*d, h, bytes, cudaMemcpyHostToDevice, st);
        return e;
    };
    SEM_CUDA_OK(c, up((void**)&s->d_link, link.data(), link.size() * sizeof(int4)));
    SEM_CUDA_OK(c, up((void**)&s->d_nrm, nrm.data(), nrm.size() * sizeof(int32_t)));
    SEM_CUDA_OK(c, up((void**)&s->d_S64, S.data(), S.size() * sizeof(double)));
    SEM_CUDA_OK(c, up((void**)&s->d_iL64, iL.data(), iL.size() * sizeof(double)));
    SEM_CUDA_OK(c, up((void**)&s->d_S32, S32.data(), S32.size() * sizeof(float)));
    SEM_CUDA_OK(c, up((void**)&s->d_iL32, iL32.data(), iL32.size() * sizeof(float)));
    SEM_CUDA_OK(c, cudaMalloc(&s->d_ext, E * m3 * sizeof(double)));
    for (int k = 0; k < 2; ++k) {
        SEM_CUDA_OK(c, cudaMalloc((void**)&s->d_W64[k], c->nL * sizeof(double)));
        SEM_CUDA_OK(c, cudaMalloc((void**)&s->d_W32[k], c->nL * sizeof(float)));
    }
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));                       // the host vectors go out of scope below
    // ---- weights: push ones through extension and combination (no solve), sum the copies, invert ----
    double* ones = nullptr;
    SEM_CUDA_OK(c, cudaMalloc((void**)&ones, c->nL * sizeof(double)));
    const unsigned vgrid = (unsigned)c->num_sms * 8;
    const unsigned egrid = (unsigned)E;
    for (int k = 0; k < 2; ++k) {
        k_fill<double><<<vgrid, 256, 0, st>>>(c->nL, 1.0, ones);
        launch_ext<double>(c, egrid, ones, nullptr, (double*)s->d_ext);
        launch_combine<double>(c, egrid, k == SEM_SCHWARZ_RAS, (const double*)s->d_ext, nullptr, ones);
        if ((rc = sem_launch_gs(c, ones, SEM_F64, /*apply_mask=*/false))) { cudaFree(ones); return rc; }
        k_inv_w<<<vgrid, 256, 0, st>>>(c->nL, ones, k == SEM_SCHWARZ_ASM, s->d_W64[k], s->d_W32[k]);
    }
    cudaError_t e = cudaStreamSynchronize(st);
    cudaFree(ones);
    if (e != cudaSuccess) return sem_fail(c, SEM_ECUDA, "sem_schwarz_setup: %s", cudaGetErrorString(e));
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

static int check(sem_ctx* c, const void* r, void* z, sem_prec prec, int kind, const char* who) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (!r || !z) return sem_fail(c, SEM_EINVAL, "%s: NULL vector", who);
    if (prec != SEM_F64 && prec != SEM_F32) return sem_fail(c, SEM_EINVAL, "%s: bad sem_prec", who);
    if (kind != SEM_SCHWARZ_ASM && kind != SEM_SCHWARZ_RAS) return sem_fail(c, SEM_EINVAL, "%s: bad sem_schwarz_kind", who);
    if (!c->sw) return sem_fail(c, SEM_ESTATE, "%s before sem_schwarz_setup", who);
    return SEM_OK;
}

extern "C" int sem_schwarz(sem_ctx* c, const void* r, void* z, sem_prec prec, sem_schwarz_kind kind) {
    int rc = check(c, r, z, prec, (int)kind, "sem_schwarz");
    if (rc) return rc;
    return sem_launch_schwarz(c, r, z, prec, (int)kind);
}

extern "C" int sem_get_schwarz(sem_ctx* c, int32_t* nbr, double* A, double* B, double* W, sem_schwarz_kind kind) {
    if (!c) return SEM_EINVAL;
    c->err.clear();
    if (!c->sw) return sem_fail(c, SEM_ESTATE, "sem_get_schwarz before sem_schwarz_setup");
    if (kind != SEM_SCHWARZ_ASM && kind != SEM_SCHWARZ_RAS) return sem_fail(c, SEM_EINVAL, "bad sem_schwarz_kind");
    sem_schwarz_data* s = c->sw;
    if (nbr) for (size_t q = 0; q < s->hnbr.size(); ++q) nbr[q] = s->hnbr[q];
    if (A) for (size_t q = 0; q < s->hA.size(); ++q) A[q] = s->hA[q];
    if (B) for (size_t q = 0; q < s->hB.size(); ++q) B[q] = s->hB[q];
    if (W) {                                       // ASM: the square root of the weight (it is applied on both sides)
        SEM_CUDA_OK(c, cudaMemcpyAsync(W, s->d_W64[kind], c->nL * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        SEM_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    }
    return SEM_OK;
}
