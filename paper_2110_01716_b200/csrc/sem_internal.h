// sem_internal.h — context struct and internal launcher declarations of libsem.so (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/sem.h"

#define SEM_MAXP 16
#define SEM_MAX_DEVICES 64      // per-device caches of launch configurations (occupancy, shared-memory opt-in)

// Elements per CTA ("group") of the Ax kernels: enough elements to fill 64 threads with one (i,j) column each.
// G is stored group-blocked so that one k-slab of one group is one contiguous chunk (one bulk copy):
//   Gs[grp][k][slot][c][j*p+i],  grp = e / epb, slot = e % epb, c = rr,rs,rt,ss,st,tt;  padded to whole groups.
__host__ __device__ inline int sem_epb(int p) { return p * p >= 64 ? 1 : (64 + p * p - 1) / (p * p); }
__host__ __device__ inline int64_t sem_g_off(int64_t e, int k, int p, int epb, int64_t slab) {
    const int64_t grp = e / epb;
    return ((grp * p + k) * epb + (e - grp * epb)) * slab;
}

struct sem_schwarz_data;            // sem_schwarz.cu
struct sem_coarse_data;             // sem_coarse.cu

struct sem_ctx {
    // ---- discretisation (a0) ----
    int64_t E = 0;
    int N = 0, p = 0;
    int64_t p3 = 0, nL = 0;
    double xi[SEM_MAXP], rho[SEM_MAXP], D[SEM_MAXP * SEM_MAXP];   // D[i*p+l] = dh_l/dr(xi_i)
    cudaStream_t stream = 0;
    int device = 0, num_sms = 148;
    // ---- mesh ----
    double* d_vert = nullptr;      // [E][8][3]
    // ---- gather-scatter maps (a1, O6) ----
    int64_t U = 0, S = 0, Us = 0;
    int32_t* d_l2u = nullptr;      // [nL]
    int32_t* d_mult = nullptr;     // [U]
    int64_t* d_seg_off = nullptr;  // [U+1]
    int32_t* d_seg_idx = nullptr;  // [nL]
    int64_t* d_uniq_gid = nullptr; // [U]
    // compressed shared-only form used by the gs kernel: unique nodes with mult > 1, ascending
    int32_t* d_sh_off = nullptr;   // [Us+1] offsets into d_sh_idx
    int32_t* d_sh_idx = nullptr;   // [S] local indices
    uint8_t* d_sh_masked = nullptr;// [Us] 1 = Dirichlet
    // pre-resolved gather-scatter records (sem_maps.cu: sem_build_gs_records), sorted by the element group that holds
    // the node's LAST (highest local index) copy, so that consecutive records touch neighbouring memory:
    //   pairs  int2 (l0 | maskbit, l1)              nodes with 2 copies; l1 = -1: only zero w[l0] (unshared Dirichlet node)
    //   quads  int4 (l0 | maskbit, l1, l2, l3 or -1) 3 or 4 copies
    //   bigs   int2 (offset into d_sh_idx, count | maskbit)   > 4 copies
    int epb = 1;
    int64_t ngroups = 0;
    int2* d_own_pair = nullptr;
    int4* d_own_quad = nullptr;
    int2* d_own_big = nullptr;
    int64_t n_pair = 0, n_quad = 0, n_big = 0;
    // chunks of whole element groups for fields that do not fit in L2 (empty: no chunking): element bounds and, per
    // record class, the first record owned by each chunk (records are sorted by owner group)
    std::vector<int64_t> chunk_e0;
    std::vector<int32_t> chunk_rec[3];
    std::vector<int32_t> grp_rec[3];         // host copy of the per-group record offsets, [ngroups + 1] per class
    // sharded solves (sem_shard.cu): the first iface_chunks chunks hold every element that touches a node shared with
    // another rank (0: the exchange starts after the whole apply); Minv / dot weights assembled over all ranks
    int iface_chunks = 0;
    double* d_Minv_g = nullptr;
    double* d_wt_g = nullptr;
    double lambda_of_shard = -1.0;
    int64_t rng_e0 = 0, rng_ne = 0;          // element range of the Ax launch in flight (sem_launch_ax_gs), 0 = all
    // Dirichlet (S14)
    bool has_mask = false;
    uint8_t* d_mask_u = nullptr;   // [U] 1 = masked unique node
    int64_t n_mask1 = 0;           // masked local nodes with mult == 1
    int32_t* d_mask1_idx = nullptr;// [n_mask1]
    // ---- geometry (a2, O3) ----
    bool geom_done = false;
    sem_gmode gmode = SEM_G_STORED;
    bool with_mass = false;
    // group-blocked slab layout (see sem_g_off above); slab stride (values per element slab) padded to 16 B
    double* d_G = nullptr;
    float* d_G32 = nullptr;        // built lazily at the first FP32 call
    double* d_B = nullptr;         // [E][p^3] rho rho rho detJ   (with_mass)
    float* d_B32 = nullptr;
    double* d_detJ = nullptr;      // [E][p^3]
    int64_t slab_f64 = 0, slab_f32 = 0;   // slab strides in elements of T
    // ---- Jacobi / PCG (a8, O7, O8) ----
    double lambda = 0.0;
    double* d_diag = nullptr;      // assembled, unmasked, local layout
    double* d_Minv = nullptr;      // mask / diag, local layout
    double* d_wt = nullptr;        // 1/mult per local node (0 at masked nodes): unique-node dot weights
    uint8_t* d_wt8 = nullptr;      // multiplicity per local node as a byte (0 at masked nodes); nullptr if some
                                   // multiplicity exceeds 255 (then the kernels read d_wt)
    bool pcg_ready = false;
    double lambda_of_diag = -1.0;  // lambda the stored diagonal was built for (-1 = none)
    double *d_r = nullptr, *d_p = nullptr, *d_w = nullptr;
    double* d_scal = nullptr;      // device scalars, see sem_pcg.cu
    int64_t scal_cap = 0;
    double* h_hist = nullptr;
    int hist_n = 0;
    // ---- p-multigrid transfer (NEXT-1, sem_transfer.cu) ----
    void* d_J = nullptr;           // interpolation matrices, one slot of SEM_MAXP^2 doubles per key = (coarse p) * 2 +
    uint64_t J_have = 0;           // (FP32 ? 1 : 0), each written once (bit `key` of J_have): graphs never see a rewrite
    float* d_Minv32 = nullptr;     // Minv rounded to FP32 for the FP32 smoother (sem_cheby.cu)
    double lambda_of_minv32 = -1.0;
    void* d_cheb4 = nullptr;       // fourth work vector of the Chebyshev-Schwarz smoother (S applied out of place)
    void* d_cheb[3] = {nullptr, nullptr, nullptr};   // r, d, w of the Chebyshev smoother (sem_cheby.cu), nL doubles each
    // element renumbering for the solver's own vectors (sem_inner.cu): a second context over the same elements sorted by
    // smallest global id, used by sem_pcg on large meshes whose element order has no locality
    sem_ctx* inner = nullptr;
    bool is_inner = false;
    int32_t* d_perm = nullptr;      // [E] inner position q holds caller element d_perm[q]
    double *d_bi = nullptr, *d_xi = nullptr;
    sem_coarse_data* coarse = nullptr;   // N = 1: assembled operator of the coarsest multigrid level (sem_coarse.cu)
    sem_schwarz_data* sw = nullptr; // NEXT-2b: face links, 1-D operator factorisations, weights (sem_schwarz_setup)
    uint64_t generation = 0;       // bumped whenever device pointers or parameters that launches capture may change
                                   // (sem_geom, sem_set_lambda): invalidates CUDA graphs recorded over this context
    // ---- CUDA graph of one sem_ax_gs application (sem_api.cu), valid for the argument set it was recorded with ----
    cudaGraphExec_t ag_exec = nullptr;
    bool ag_exec_or_seen = false, ag_capturable = false;
    const void* ag_u = nullptr;
    void* ag_w = nullptr;
    int ag_prec = -1, ag_variant = 0;
    double ag_lambda = 0.0;
    uint64_t ag_gen = 0;
    // ---- misc ----
    int ax_variant = 0;
    int fdm_variant = 0;           // sem_set_variant(100 + v): 0 = scalar local-solve kernels, 1 = FP32 tensor-core kernel
    std::string err;
};

int sem_fail(sem_ctx* c, int code, const char* fmt, ...);
#define SEM_CUDA_OK(c, expr)                                                                          \
    do {                                                                                              \
        cudaError_t e__ = (expr);                                                                     \
        if (e__ != cudaSuccess)                                                                       \
            return sem_fail((c), e__ == cudaErrorMemoryAllocation ? SEM_ENOMEM : SEM_ECUDA, "%s: %s", \
                            #expr, cudaGetErrorString(e__));                                          \
    } while (0)

// sem_gll.cpp
void sem_gll_tables(int N, double* xi, double* rho, double* D);
// sem_maps.cu
int sem_build_maps(sem_ctx* c, const int64_t* gid_any, const uint8_t* dirichlet_host);
int sem_build_gs_records(sem_ctx* c);
// sem_geom.cu
int sem_build_geom(sem_ctx* c, const double* node_xyz_host);
int sem_build_g32(sem_ctx* c);
int sem_ensure_G(sem_ctx* c);       // recompute mode keeps no stored G: rebuilt for the diagonal / the accessor
void sem_release_G(sem_ctx* c);
int sem_build_diag(sem_ctx* c);
int sem_geom_export(sem_ctx* c, double* G_host, double* detJ_host);
// sem_ax.cu
int sem_launch_ax(sem_ctx* c, const void* u, void* w, sem_prec prec, double lambda, double* dot_out,
                  const int* skip_flag);
int sem_launch_ax_gs(sem_ctx* c, const void* u, void* w, sem_prec prec, double lambda, double* dot_out,
                     const int* skip_flag);
int sem_launch_ax_gs_chunks(sem_ctx* c, const void* u, void* w, sem_prec prec, double lambda, double* dot_out,
                            const int* skip_flag, int q0, int q1);      // a3-a7: operator kernel + gather-scatter kernel
int sem_launch_ax_many(sem_ctx* c, const void* u, void* w, int nf, int64_t stride, sem_prec prec, double lambda,
                       double* dot_out, int64_t dot_stride, const int* skip_flag);
// sem_gs.cu
int sem_launch_gs(sem_ctx* c, void* w, sem_prec prec, bool apply_mask, const int* skip_flag = nullptr);
int sem_launch_gs_range(sem_ctx* c, void* w, sem_prec prec, bool apply_mask, const int* skip_flag, int chunk);
// sem_shard.cu
int sem_hooks_ok(sem_ctx* c, const sem_shard_hooks* h, const char* who);
int sem_launch_ax_gs_sharded(sem_ctx* c, const void* u, void* w, sem_prec prec, double lambda, double* dot_out,
                             const int* skip_flag, const sem_shard_hooks* h);
int sem_shard_build_diag(sem_ctx* c, const sem_shard_hooks* h);
void sem_set_chunk_groups(sem_ctx* c, const std::vector<int64_t>& group_bounds);
void sem_default_chunks(sem_ctx* c, int64_t first_groups);
int sem_launch_gs_many(sem_ctx* c, void* w, int nf, int64_t stride, sem_prec prec, bool apply_mask,
                       const int* skip_flag = nullptr);
// sem_api.cu
int sem_launch_gs_fields(sem_ctx* c, void* w, int nf, int64_t stride, sem_prec prec, bool mask, const int* skip);
// sem_api.cu
int sem_launch_gs_fields(sem_ctx* c, void* w, int nf, int64_t stride, sem_prec prec, bool mask, const int* skip);
// sem_api.cu / sem_inner.cu
int sem_mesh_setup_impl(sem_ctx** out, int64_t E, int N, const double* vertex_xyz, const int64_t* gid,
                        const uint8_t* dirichlet, void* cuda_stream, bool is_inner);
int sem_inner_build(sem_ctx* c, const double* node_xyz_host);
void sem_inner_free(sem_ctx* c);
int sem_inner_pcg(sem_ctx* c, const double* b, double* x, double tol, int maxit, int* iters_out, double* relres_out);
// sem_fdm.cu
int sem_launch_fdm_schwarz(sem_ctx* c, int m, const void* S, const void* invL, const void* r, const int4* link,
                           const int32_t* nrm, const void* W, void* z, sem_prec prec);
// sem_coarse.cu
int sem_coarse_build(sem_ctx* c);
void sem_coarse_free(sem_ctx* c);
bool sem_coarse_is_current(const sem_ctx* c);     // built for the context's current lambda
int sem_coarse_cheby(sem_ctx* c, const void* b, void* x, int order, double lmin, double lmax, bool zero_guess,
                     sem_prec prec);
// sem_schwarz.cu
void sem_schwarz_free(sem_ctx* c);
int sem_launch_schwarz(sem_ctx* c, const void* r, void* z, sem_prec prec, int kind);   // z may alias r
// sem_transfer.cu
int sem_launch_transfer(sem_ctx* coarse, sem_ctx* fine, const void* in, void* out, sem_prec prec, sem_transfer_dir dir,
                        const void* in_minus, const double* wt);
