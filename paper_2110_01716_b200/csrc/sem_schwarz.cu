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

// b~: one thread per block position
template <typename T>
__global__ void __launch_bounds__(256) k_schwarz_ext(int64_t E, int p, const int4* __restrict__ link,
                                                     const int32_t* __restrict__ nrm, const T* __restrict__ r,
                                                     const T* __restrict__ pre, T* __restrict__ ext) {
    const int m = p + 2, m3 = m * m * m, p3 = p * p * p;
    for (int64_t e = blockIdx.x; e < E; e += gridDim.x) {
        for (int q = threadIdx.x; q < m3; q += blockDim.x) {
            const int a = q % m, b = (q / m) % m, c = q / (m * m);
            const int ga = (a == 0 || a == m - 1), gb = (b == 0 || b == m - 1), gc = (c == 0 || c == m - 1);
            T v = T(0);
            if (ga + gb + gc == 0) {
                const int64_t l = e * p3 + ((c - 1) * p + (b - 1)) * p + (a - 1);
                v = pre ? pre[l] * r[l] : r[l];
            } else if (ga + gb + gc == 1) {
                const int axis = ga ? 0 : (gb ? 1 : 2);
                const int side = (ga ? a : (gb ? b : c)) != 0;
                const int fa = axis == 0 ? b - 1 : a - 1, fb = axis == 2 ? b - 1 : c - 1;
                const int4 lk = link[e * 6 + 2 * axis + side];
                if (lk.x >= 0) {
                    const int32_t nf = nrm[e * 6 + 2 * axis + side];
                    const int na = nf & 3, ns = nf >> 2;
                    int stride = 1;
                    for (int t = 0; t < na; ++t) stride *= p;
                    const int l = lk.y + fa * lk.z + fb * lk.w + (ns ? -stride : stride);      // one layer in
                    v = pre ? pre[(int64_t)lk.x * p3 + l] * r[(int64_t)lk.x * p3 + l] : r[(int64_t)lk.x * p3 + l];
                }
            }
            ext[e * m3 + q] = v;
        }
    }
}

// z_L = W (own part of u~ + ghost layers of the face neighbours), one thread per local node
template <typename T, bool RESTRICTED>
__global__ void __launch_bounds__(256) k_schwarz_combine(int64_t E, int p, const int4* __restrict__ link,
                                                         const int32_t* __restrict__ nrm, const T* __restrict__ ext,
                                                         const T* __restrict__ W, T* __restrict__ z) {
    const int m = p + 2, m3 = m * m * m, p3 = p * p * p, N = p - 1;
    for (int64_t e = blockIdx.x; e < E; e += gridDim.x) {
        for (int l = threadIdx.x; l < p3; l += blockDim.x) {
            const int i = l % p, j = (l / p) % p, k = l / (p * p);
            T v = ext[e * m3 + ((k + 1) * m + (j + 1)) * m + (i + 1)];
            if (!RESTRICTED) {
                const int co[3] = {i, j, k};
#pragma unroll
                for (int axis = 0; axis < 3; ++axis)
#pragma unroll
                    for (int side = 0; side < 2; ++side) {
                        if (co[axis] != (side ? N - 1 : 1)) continue;          // not in the one-layer-in plane of this face
                        const int4 lk = link[e * 6 + 2 * axis + side];
                        if (lk.x < 0) continue;
                        const int fa = axis == 0 ? j : i, fb = axis == 2 ? j : k;
                        const int ln = lk.y + fa * lk.z + fb * lk.w;            // neighbour's face node behind mine
                        const int32_t nf = nrm[e * 6 + 2 * axis + side];
                        const int na = nf & 3, ns = nf >> 2;
                        int ci = ln % p + 1, cj = (ln / p) % p + 1, ck = ln / (p * p) + 1;   // block coordinates
                        if (na == 0) ci += ns ? 1 : -1;                          // one step OUT of the neighbour: its ghost
                        else if (na == 1) cj += ns ? 1 : -1;
                        else ck += ns ? 1 : -1;
                        v += ext[(int64_t)lk.x * m3 + (ck * m + cj) * m + ci];
                    }
            }
            z[e * p3 + l] = W ? W[e * p3 + l] * v : v;
        }
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

template <typename T>
int apply(sem_ctx* c, const T* r, T* z, int kind) {
    sem_schwarz_data* s = c->sw;
    const sem_prec prec = sizeof(T) == 8 ? SEM_F64 : SEM_F32;
    const T* S = sizeof(T) == 8 ? (const T*)s->d_S64 : (const T*)s->d_S32;
    const T* iL = sizeof(T) == 8 ? (const T*)s->d_iL64 : (const T*)s->d_iL32;
    const T* W = sizeof(T) == 8 ? (const T*)s->d_W64[kind] : (const T*)s->d_W32[kind];
    T* ext = (T*)s->d_ext;
    const unsigned grid = (unsigned)(c->E < (int64_t)c->num_sms * 8 ? c->E : (int64_t)c->num_sms * 8);
    k_schwarz_ext<T><<<grid, 256, 0, c->stream>>>(c->E, c->p, s->d_link, s->d_nrm, r,
                                                  kind == SEM_SCHWARZ_ASM ? W : (const T*)nullptr, ext);
    int rc = sem_fdm_apply(c, s->m, S, iL, ext, ext, prec);
    if (rc) return rc;
    if (kind == SEM_SCHWARZ_RAS)
        k_schwarz_combine<T, true><<<grid, 256, 0, c->stream>>>(c->E, c->p, s->d_link, s->d_nrm, ext, W, z);
    else
        k_schwarz_combine<T, false><<<grid, 256, 0, c->stream>>>(c->E, c->p, s->d_link, s->d_nrm, ext, W, z);
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
    const unsigned egrid = (unsigned)(E < (int64_t)c->num_sms * 8 ? E : (int64_t)c->num_sms * 8);
    for (int k = 0; k < 2; ++k) {
        k_fill<double><<<vgrid, 256, 0, st>>>(c->nL, 1.0, ones);
        k_schwarz_ext<double><<<egrid, 256, 0, st>>>(E, p, s->d_link, s->d_nrm, ones, nullptr, (double*)s->d_ext);
        if (k == SEM_SCHWARZ_RAS)
            k_schwarz_combine<double, true><<<egrid, 256, 0, st>>>(E, p, s->d_link, s->d_nrm, (const double*)s->d_ext, nullptr, ones);
        else
            k_schwarz_combine<double, false><<<egrid, 256, 0, st>>>(E, p, s->d_link, s->d_nrm, (const double*)s->d_ext, nullptr, ones);
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
