// sem_maps.cu — a1 (setup): canonical gather-scatter maps from one global id per local node.
// P:121 "the user (or code) simply provides a global ID for each vertex"; contract O6:
//   uniq_gid = distinct gids ascending; l2u[l] = rank of gid[l]; mult[g] = copies; seg_off = exclusive scan of mult;
//   seg_idx = local indices ordered by (gid, l) ascending, i.e. a STABLE sort of l by gid.
// All integer work, bit-exact.  The sort and the scans are CUB device primitives (setup, untimed); everything on
// the timed path (sem_gs.cu) is hand-written.
#include <stdlib.h>

#include <cub/cub.cuh>

#include "sem_internal.h"

namespace {

__global__ void k_iota_minmax(int64_t n, const int64_t* __restrict__ gid, int32_t* __restrict__ vals,
                              unsigned long long* __restrict__ maxgid, int* __restrict__ neg) {
    int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    unsigned long long mx = 0;
    int bad = 0;
    for (; t < n; t += stride) {
        const int64_t g = gid[t];
        vals[t] = (int32_t)t;
        if (g < 0) bad = 1; else if ((unsigned long long)g > mx) mx = (unsigned long long)g;
    }
    for (int o = 16; o; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, mx, o);
        mx = other > mx ? other : mx;
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMax(maxgid, mx);
        if (bad) atomicOr(neg, 1);
    }
}

// head[q] = 1 where a new gid starts in the sorted key list
__global__ void k_heads(int64_t n, const int64_t* __restrict__ keys, int32_t* __restrict__ head) {
    const int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (q < n) head[q] = (q == 0 || keys[q] != keys[q - 1]) ? 1 : 0;
}

// rank[q] = inclusive scan of head (1-based unique index).  Scatter the maps.
__global__ void k_scatter_maps(int64_t n, const int64_t* __restrict__ keys, const int32_t* __restrict__ sorted_l,
                               const int32_t* __restrict__ rank, int32_t* __restrict__ l2u,
                               int64_t* __restrict__ uniq_gid, int64_t* __restrict__ seg_off, int64_t U) {
    const int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (q >= n) return;
    const int32_t g = rank[q] - 1;
    l2u[sorted_l[q]] = g;
    if (q == 0 || rank[q] != rank[q - 1]) { uniq_gid[g] = keys[q]; seg_off[g] = q; }
    if (q == n - 1) seg_off[U] = n;
}

__global__ void k_mult(int64_t U, const int64_t* __restrict__ seg_off, int32_t* __restrict__ mult,
                       int32_t* __restrict__ is_shared, int32_t* __restrict__ shared_cnt) {
    const int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (g >= U) return;
    const int32_t m = (int32_t)(seg_off[g + 1] - seg_off[g]);
    mult[g] = m;
    is_shared[g] = m > 1 ? 1 : 0;
    shared_cnt[g] = m > 1 ? m : 0;
}

// unique-node mask = OR over copies (S14)
__global__ void k_mask_u(int64_t U, const int64_t* __restrict__ seg_off, const int32_t* __restrict__ seg_idx,
                         const uint8_t* __restrict__ dir_l, uint8_t* __restrict__ mask_u) {
    const int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (g >= U) return;
    uint8_t m = 0;
    for (int64_t q = seg_off[g]; q < seg_off[g + 1]; ++q) m |= dir_l[seg_idx[q]] ? 1 : 0;
    mask_u[g] = m;
}

// compressed shared-only form: s = (exclusive scan of is_shared)[g]; sh_off[s] = (exclusive scan of shared_cnt)[g]
__global__ void k_compress_shared(int64_t U, const int64_t* __restrict__ seg_off, const int32_t* __restrict__ seg_idx,
                                  const int32_t* __restrict__ is_shared, const int32_t* __restrict__ sh_rank_ex,
                                  const int32_t* __restrict__ sh_cnt_ex, const uint8_t* __restrict__ mask_u,
                                  int32_t* __restrict__ sh_off, int32_t* __restrict__ sh_idx,
                                  uint8_t* __restrict__ sh_masked) {
    const int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (g >= U || !is_shared[g]) return;
    const int32_t s = sh_rank_ex[g];
    const int32_t o = sh_cnt_ex[g];
    sh_off[s] = o;
    sh_masked[s] = mask_u ? mask_u[g] : 0;
    const int64_t q0 = seg_off[g];
    const int32_t m = (int32_t)(seg_off[g + 1] - q0);
    for (int32_t r = 0; r < m; ++r) sh_idx[o + r] = seg_idx[q0 + r];
}

// flag for local nodes that are masked and not shared (the gs kernel zeroes shared masked nodes itself)
__global__ void k_mask1_flag(int64_t n, const int32_t* __restrict__ l2u, const int32_t* __restrict__ mult,
                             const uint8_t* __restrict__ mask_u, int32_t* __restrict__ flag) {
    const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (l >= n) return;
    const int32_t g = l2u[l];
    flag[l] = (mask_u[g] && mult[g] == 1) ? 1 : 0;
}

__global__ void k_mask1_fill(int64_t n, const int32_t* __restrict__ flag, const int32_t* __restrict__ ex,
                             int32_t* __restrict__ out) {
    const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (l < n && flag[l]) out[ex[l]] = (int32_t)l;
}

struct Tmp {   // frees device scratch on every exit path
    void* ptrs[40]; int n = 0;
    template <typename T> cudaError_t alloc(T** p, size_t count) {
        cudaError_t e = cudaMalloc((void**)p, (count ? count : 1) * sizeof(T));
        if (e == cudaSuccess) ptrs[n++] = *p;
        return e;
    }
    ~Tmp() { for (int i = 0; i < n; ++i) cudaFree(ptrs[i]); }
};

inline unsigned nblk(int64_t n, int t = 256) { return (unsigned)((n + t - 1) / t); }

}  // namespace

int sem_build_maps(sem_ctx* c, const int64_t* gid_any, const uint8_t* dirichlet_host) {
    const int64_t n = c->nL;
    cudaStream_t st = c->stream;
    Tmp tmp;
    // ---- gid on the device ----
    cudaPointerAttributes attr;
    bool on_device = false;
    if (cudaPointerGetAttributes(&attr, gid_any) == cudaSuccess)
        on_device = (attr.type == cudaMemoryTypeDevice || attr.type == cudaMemoryTypeManaged);
    else
        cudaGetLastError();
    int64_t* d_gid = nullptr;
    if (on_device) d_gid = const_cast<int64_t*>(gid_any);
    else {
        SEM_CUDA_OK(c, tmp.alloc(&d_gid, n));
        SEM_CUDA_OK(c, cudaMemcpyAsync(d_gid, gid_any, n * sizeof(int64_t), cudaMemcpyHostToDevice, st));
    }
    // ---- validate, find the key width ----
    int32_t *d_vals_in = nullptr, *d_vals_out = nullptr;
    int64_t* d_keys_out = nullptr;
    unsigned long long* d_max = nullptr;
    int* d_neg = nullptr;
    SEM_CUDA_OK(c, tmp.alloc(&d_vals_in, n));
    SEM_CUDA_OK(c, tmp.alloc(&d_keys_out, n));
    SEM_CUDA_OK(c, tmp.alloc(&d_max, 1));
    SEM_CUDA_OK(c, tmp.alloc(&d_neg, 1));
    SEM_CUDA_OK(c, cudaMemsetAsync(d_max, 0, sizeof(*d_max), st));
    SEM_CUDA_OK(c, cudaMemsetAsync(d_neg, 0, sizeof(*d_neg), st));
    k_iota_minmax<<<c->num_sms * 8, 256, 0, st>>>(n, d_gid, d_vals_in, d_max, d_neg);
    unsigned long long h_max = 0;
    int h_neg = 0;
    SEM_CUDA_OK(c, cudaMemcpyAsync(&h_max, d_max, sizeof(h_max), cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaMemcpyAsync(&h_neg, d_neg, sizeof(h_neg), cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    if (h_neg) return sem_fail(c, SEM_EINVAL, "negative global id (S11: gids must be >= 0)");
    int end_bit = 1;
    while (end_bit < 63 && (h_max >> end_bit)) ++end_bit;
    // ---- stable sort of (gid, l) ----
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_seg_idx, n * sizeof(int32_t)));
    d_vals_out = c->d_seg_idx;
    size_t tb = 0;
    SEM_CUDA_OK(c, cub::DeviceRadixSort::SortPairs(nullptr, tb, d_gid, d_keys_out, d_vals_in, d_vals_out, n, 0,
                                                    end_bit, st));
    void* d_tmp = nullptr;
    SEM_CUDA_OK(c, tmp.alloc((char**)&d_tmp, tb));
    SEM_CUDA_OK(c, cub::DeviceRadixSort::SortPairs(d_tmp, tb, d_gid, d_keys_out, d_vals_in, d_vals_out, n, 0, end_bit,
                                                    st));
    // ---- ranks ----
    int32_t* d_rank = d_vals_in;   // reuse: iota no longer needed
    k_heads<<<nblk(n), 256, 0, st>>>(n, d_keys_out, d_rank);
    size_t tb2 = 0;
    SEM_CUDA_OK(c, cub::DeviceScan::InclusiveSum(nullptr, tb2, d_rank, d_rank, n, st));
    void* d_tmp2 = d_tmp;
    if (tb2 > tb) SEM_CUDA_OK(c, tmp.alloc((char**)&d_tmp2, tb2));
    SEM_CUDA_OK(c, cub::DeviceScan::InclusiveSum(d_tmp2, tb2, d_rank, d_rank, n, st));
    int32_t h_U = 0;
    SEM_CUDA_OK(c, cudaMemcpyAsync(&h_U, d_rank + (n - 1), sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    const int64_t U = h_U;
    c->U = U;
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_l2u, n * sizeof(int32_t)));
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_uniq_gid, U * sizeof(int64_t)));
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_seg_off, (U + 1) * sizeof(int64_t)));
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_mult, U * sizeof(int32_t)));
    k_scatter_maps<<<nblk(n), 256, 0, st>>>(n, d_keys_out, c->d_seg_idx, d_rank, c->d_l2u, c->d_uniq_gid, c->d_seg_off, U);
    // ---- multiplicities, shared-only compressed form ----
    int32_t *d_is_sh = nullptr, *d_sh_cnt = nullptr;
    SEM_CUDA_OK(c, tmp.alloc(&d_is_sh, U + 1));
    SEM_CUDA_OK(c, tmp.alloc(&d_sh_cnt, U + 1));
    SEM_CUDA_OK(c, cudaMemsetAsync(d_is_sh + U, 0, sizeof(int32_t), st));
    SEM_CUDA_OK(c, cudaMemsetAsync(d_sh_cnt + U, 0, sizeof(int32_t), st));
    k_mult<<<nblk(U), 256, 0, st>>>(U, c->d_seg_off, c->d_mult, d_is_sh, d_sh_cnt);
    int32_t *d_is_sh_ex = nullptr, *d_sh_cnt_ex = nullptr;
    SEM_CUDA_OK(c, tmp.alloc(&d_is_sh_ex, U + 1));
    SEM_CUDA_OK(c, tmp.alloc(&d_sh_cnt_ex, U + 1));
    size_t tb3 = 0;
    SEM_CUDA_OK(c, cub::DeviceScan::ExclusiveSum(nullptr, tb3, d_is_sh, d_is_sh_ex, U + 1, st));
    void* d_tmp3 = d_tmp2;
    if (tb3 > (tb2 > tb ? tb2 : tb)) SEM_CUDA_OK(c, tmp.alloc((char**)&d_tmp3, tb3));
    SEM_CUDA_OK(c, cub::DeviceScan::ExclusiveSum(d_tmp3, tb3, d_is_sh, d_is_sh_ex, U + 1, st));
    SEM_CUDA_OK(c, cub::DeviceScan::ExclusiveSum(d_tmp3, tb3, d_sh_cnt, d_sh_cnt_ex, U + 1, st));
    int32_t h_Us = 0, h_S = 0;
    SEM_CUDA_OK(c, cudaMemcpyAsync(&h_Us, d_is_sh_ex + U, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaMemcpyAsync(&h_S, d_sh_cnt_ex + U, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    c->Us = h_Us;
    c->S = h_S;
    // ---- Dirichlet mask ----
    uint8_t* d_dir = nullptr;
    c->has_mask = dirichlet_host != nullptr;
    if (c->has_mask) {
        SEM_CUDA_OK(c, tmp.alloc(&d_dir, n));
        SEM_CUDA_OK(c, cudaMemcpyAsync(d_dir, dirichlet_host, n, cudaMemcpyHostToDevice, st));
        SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_mask_u, U));
        k_mask_u<<<nblk(U), 256, 0, st>>>(U, c->d_seg_off, c->d_seg_idx, d_dir, c->d_mask_u);
    }
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_sh_off, (c->Us + 1) * sizeof(int32_t)));
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_sh_idx, (c->S ? c->S : 1) * sizeof(int32_t)));
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_sh_masked, c->Us ? c->Us : 1));
    k_compress_shared<<<nblk(U), 256, 0, st>>>(U, c->d_seg_off, c->d_seg_idx, d_is_sh, d_is_sh_ex, d_sh_cnt_ex,
                                                c->d_mask_u, c->d_sh_off, c->d_sh_idx, c->d_sh_masked);
    SEM_CUDA_OK(c, cudaMemcpyAsync(c->d_sh_off + c->Us, &h_S, sizeof(int32_t), cudaMemcpyHostToDevice, st));
    if (c->has_mask) {
        int32_t* d_flag = d_rank;           // reuse [n]
        int32_t* d_ex = nullptr;
        SEM_CUDA_OK(c, tmp.alloc(&d_ex, n + 1));
        k_mask1_flag<<<nblk(n), 256, 0, st>>>(n, c->d_l2u, c->d_mult, c->d_mask_u, d_flag);
        size_t tb4 = 0;
        SEM_CUDA_OK(c, cub::DeviceScan::ExclusiveSum(nullptr, tb4, d_flag, d_ex, n, st));
        void* d_tmp4 = nullptr;
        SEM_CUDA_OK(c, tmp.alloc((char**)&d_tmp4, tb4));
        SEM_CUDA_OK(c, cub::DeviceScan::ExclusiveSum(d_tmp4, tb4, d_flag, d_ex, n, st));
        int32_t last_ex = 0, last_flag = 0;
        SEM_CUDA_OK(c, cudaMemcpyAsync(&last_ex, d_ex + (n - 1), sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        SEM_CUDA_OK(c, cudaMemcpyAsync(&last_flag, d_flag + (n - 1), sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        SEM_CUDA_OK(c, cudaStreamSynchronize(st));
        c->n_mask1 = (int64_t)last_ex + last_flag;
        SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_mask1_idx, (c->n_mask1 ? c->n_mask1 : 1) * sizeof(int32_t)));
        k_mask1_fill<<<nblk(n), 256, 0, st>>>(n, d_flag, d_ex, c->d_mask1_idx);
    }
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// Pre-resolved gather-scatter records (see sem_internal.h / sem_gs.cu): every shared node becomes one fixed-format
// record (pair / quad / big) holding the local indices of its copies in ascending order (O5: the oracle's summation
// order), and the records are sorted by the element group of the node's last copy.  Unshared Dirichlet nodes ride
// along as "pairs" with no partner.  Integer work only; setup, untimed.
// ---------------------------------------------------------------------------------------------------------------
namespace {

constexpr uint32_t OWN_MASKBIT = 0x80000000u;

__device__ __forceinline__ int32_t grp_of(int32_t l, int32_t group_nodes) { return l / group_nodes; }

// entry id t: t < Us a shared node, else unshared masked node t - Us.  key = owner group * 4 + class.
__global__ void k_own_keys(int32_t Us, int32_t n_mask1, int32_t group_nodes, int32_t ng,
                           const int32_t* __restrict__ sh_off, const int32_t* __restrict__ sh_idx,
                           const int32_t* __restrict__ mask1_idx, uint32_t* __restrict__ keys,
                           int32_t* __restrict__ vals, int32_t* __restrict__ Hk, int32_t* __restrict__ Hc) {
    const int32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= Us + n_mask1) return;
    int32_t g, cls;
    if (t < Us) {
        const int32_t b = sh_off[t], e = sh_off[t + 1];
        g = grp_of(sh_idx[e - 1], group_nodes);
        cls = (e - b) <= 2 ? 0 : (e - b) <= 4 ? 1 : 2;
    } else {
        g = grp_of(mask1_idx[t - Us], group_nodes);
        cls = 0;
    }
    keys[t] = (uint32_t)g * 4u + (uint32_t)cls;
    vals[t] = t;
    atomicAdd(&Hk[g * 4 + cls], 1);
    atomicAdd(&Hc[(int64_t)cls * (ng + 1) + g], 1);
}

__global__ void k_own_fill(int32_t n_ent, int32_t Us, int32_t ng, const uint32_t* __restrict__ keys,
                           const int32_t* __restrict__ vals, const int32_t* __restrict__ KS,
                           const int32_t* __restrict__ offc, const int32_t* __restrict__ sh_off,
                           const int32_t* __restrict__ sh_idx, const uint8_t* __restrict__ sh_masked,
                           const int32_t* __restrict__ mask1_idx, int2* __restrict__ pairs, int4* __restrict__ quads,
                           int2* __restrict__ bigs) {
    const int32_t q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n_ent) return;
    const uint32_t key = keys[q];
    const int32_t g = (int32_t)(key >> 2), cls = (int32_t)(key & 3u), id = vals[q];
    const int32_t pos = offc[(int64_t)cls * (ng + 1) + g] + (q - KS[key]);
    if (id >= Us) {                                   // unshared Dirichlet node: zero it
        pairs[pos] = make_int2((int32_t)((uint32_t)mask1_idx[id - Us] | OWN_MASKBIT), -1);
        return;
    }
    const int32_t b = sh_off[id], cnt = sh_off[id + 1] - b;
    const uint32_t mbit = (sh_masked && sh_masked[id]) ? OWN_MASKBIT : 0u;
    if (cls == 0) pairs[pos] = make_int2((int32_t)((uint32_t)sh_idx[b] | mbit), sh_idx[b + 1]);
    else if (cls == 1)
        quads[pos] = make_int4((int32_t)((uint32_t)sh_idx[b] | mbit), sh_idx[b + 1], sh_idx[b + 2],
                               cnt == 4 ? sh_idx[b + 3] : -1);
    else bigs[pos] = make_int2(b, (int32_t)((uint32_t)cnt | mbit));
}

template <typename T>
int ex_scan(sem_ctx* c, Tmp& tmp, const T* in, T* out, int64_t n) {
    size_t tb = 0;
    SEM_CUDA_OK(c, cub::DeviceScan::ExclusiveSum(nullptr, tb, in, out, n, c->stream));
    void* d = nullptr;
    SEM_CUDA_OK(c, cudaMalloc(&d, tb ? tb : 1));
    cudaError_t e = cub::DeviceScan::ExclusiveSum(d, tb, in, out, n, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(d);
    if (e != cudaSuccess) return sem_fail(c, SEM_ECUDA, "scan: %s", cudaGetErrorString(e));
    return SEM_OK;
}

}  // namespace

// chunk table from ascending group bounds (first = 0, last = ngroups); fewer than 2 chunks: no chunking
void sem_set_chunk_groups(sem_ctx* c, const std::vector<int64_t>& gb) {
    c->chunk_e0.clear();
    for (int cls = 0; cls < 3; ++cls) c->chunk_rec[cls].clear();
    if (gb.size() < 3) return;
    for (int64_t g0 : gb) {
        c->chunk_e0.push_back(g0 * c->epb < c->E ? g0 * c->epb : c->E);
        for (int cls = 0; cls < 3; ++cls) c->chunk_rec[cls].push_back(c->grp_rec[cls][(size_t)g0]);
    }
}

// chunks for fields larger than L2: 64 MB of FP64 field per chunk (measured best at 64^3 elements, N = 7: 48-64 MB;
// smaller chunks pay the operator's ramp and tail per launch), only when there are at least 2 of them.  first_groups
// > 0 (sem_shard_set_interface): the first chunk is exactly those groups, the rest is cut the same way.
void sem_default_chunks(sem_ctx* c, int64_t first_groups) {
    const int64_t ng = c->ngroups;
    int64_t cg = (int64_t)((64.0 * 1024 * 1024) / (8.0 * (double)(c->epb * c->p3)));
    if (cg < 1) cg = 1;
    if (const char* env = getenv("SEM_CHUNK_GROUPS")) cg = atoll(env) > 0 ? atoll(env) : ng + 1;   // tests
    std::vector<int64_t> gb;
    gb.push_back(0);
    if (first_groups > 0 && first_groups < ng) gb.push_back(first_groups);
    const int64_t g_from = gb.back(), rest = ng - g_from;
    const int64_t nch = (rest + cg - 1) / cg;
    if (nch >= 2)
        for (int64_t q = 1; q < nch; ++q) gb.push_back(g_from + q * cg);
    gb.push_back(ng);
    sem_set_chunk_groups(c, gb);
}

int sem_build_gs_records(sem_ctx* c) {
    cudaStream_t st = c->stream;
    const int32_t ng = (int32_t)c->ngroups;
    const int32_t group_nodes = (int32_t)(c->epb * c->p3);
    const int32_t Us = (int32_t)c->Us, nm1 = (int32_t)(c->has_mask ? c->n_mask1 : 0);
    const int32_t n_ent = Us + nm1;
    int rc;
    Tmp tmp;
    // ---- entries by (owner group, class) ----
    uint32_t *d_keys = nullptr, *d_keys_s = nullptr;
    int32_t *d_vals = nullptr, *d_vals_s = nullptr, *d_Hk = nullptr, *d_KS = nullptr, *d_Hc = nullptr, *d_offc = nullptr;
    SEM_CUDA_OK(c, tmp.alloc(&d_keys, n_ent));
    SEM_CUDA_OK(c, tmp.alloc(&d_keys_s, n_ent));
    SEM_CUDA_OK(c, tmp.alloc(&d_vals, n_ent));
    SEM_CUDA_OK(c, tmp.alloc(&d_vals_s, n_ent));
    const int64_t nk = (int64_t)ng * 4 + 1, nc = 3 * ((int64_t)ng + 1);
    SEM_CUDA_OK(c, tmp.alloc(&d_Hk, nk));
    SEM_CUDA_OK(c, tmp.alloc(&d_KS, nk));
    SEM_CUDA_OK(c, tmp.alloc(&d_Hc, nc));
    SEM_CUDA_OK(c, tmp.alloc(&d_offc, nc));
    SEM_CUDA_OK(c, cudaMemsetAsync(d_Hk, 0, nk * sizeof(int32_t), st));
    SEM_CUDA_OK(c, cudaMemsetAsync(d_Hc, 0, nc * sizeof(int32_t), st));
    int32_t h_tot[3] = {0, 0, 0};
    if (n_ent > 0) {
        k_own_keys<<<nblk(n_ent), 256, 0, st>>>(Us, nm1, group_nodes, ng, c->d_sh_off, c->d_sh_idx, c->d_mask1_idx,
                                                d_keys, d_vals, d_Hk, d_Hc);
        int end_bit = 1;
        while (end_bit < 32 && (((uint64_t)ng * 4) >> end_bit)) ++end_bit;
        size_t tb = 0;
        SEM_CUDA_OK(c, cub::DeviceRadixSort::SortPairs(nullptr, tb, d_keys, d_keys_s, d_vals, d_vals_s, n_ent, 0,
                                                        end_bit, st));
        void* d_tmp = nullptr;
        SEM_CUDA_OK(c, tmp.alloc((char**)&d_tmp, tb));
        SEM_CUDA_OK(c, cub::DeviceRadixSort::SortPairs(d_tmp, tb, d_keys, d_keys_s, d_vals, d_vals_s, n_ent, 0, end_bit,
                                                        st));
    }
    if ((rc = ex_scan(c, tmp, d_Hk, d_KS, nk))) return rc;
    for (int cls = 0; cls < 3; ++cls)       // each class row ends with a zero: the scan leaves the class total there
        if ((rc = ex_scan(c, tmp, d_Hc + cls * ((int64_t)ng + 1), d_offc + cls * ((int64_t)ng + 1), (int64_t)ng + 1)))
            return rc;
    for (int cls = 0; cls < 3; ++cls)
        SEM_CUDA_OK(c, cudaMemcpyAsync(&h_tot[cls], d_offc + cls * ((int64_t)ng + 1) + ng, sizeof(int32_t),
                                       cudaMemcpyDeviceToHost, st));
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    c->n_pair = h_tot[0]; c->n_quad = h_tot[1]; c->n_big = h_tot[2];
    // host copy of the per-group record offsets (3 classes x (ng + 1)): chunk tables are cut from it
    for (int cls = 0; cls < 3; ++cls) {
        c->grp_rec[cls].assign((size_t)ng + 1, 0);
        SEM_CUDA_OK(c, cudaMemcpy(c->grp_rec[cls].data(), d_offc + cls * ((int64_t)ng + 1), ((size_t)ng + 1) * sizeof(int32_t),
                                  cudaMemcpyDeviceToHost));
    }
    sem_default_chunks(c, 0);
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_own_pair, (size_t)(c->n_pair ? c->n_pair : 1) * sizeof(int2)));
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_own_quad, (size_t)(c->n_quad ? c->n_quad : 1) * sizeof(int4)));
    SEM_CUDA_OK(c, cudaMalloc((void**)&c->d_own_big, (size_t)(c->n_big ? c->n_big : 1) * sizeof(int2)));
    if (n_ent > 0)
        k_own_fill<<<nblk(n_ent), 256, 0, st>>>(n_ent, Us, ng, d_keys_s, d_vals_s, d_KS, d_offc, c->d_sh_off, c->d_sh_idx,
                                                c->has_mask ? c->d_sh_masked : nullptr, c->d_mask1_idx, c->d_own_pair,
                                                c->d_own_quad, c->d_own_big);
    SEM_CUDA_OK(c, cudaStreamSynchronize(st));
    SEM_CUDA_OK(c, cudaGetLastError());
    return SEM_OK;
}
