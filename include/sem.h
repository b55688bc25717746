/* sem.h — C ABI of libsem.so: the matrix-free spectral-element Poisson/Helmholtz hot path of arXiv 2110.01716
 * (Nek5000/RS) on one NVIDIA B200 (sm_100a).
 *
 *      w = M Q Q^T (D^T G D + lambda B) u          and the Jacobi-PCG loop that drives it.
 *
 * Citations: "P:nn" = line nn of PAPER.md; "O#/S#" = the readings listed in DESIGN.md.
 *
 * Conventions (S4): p = N+1 GLL points per direction; an element's nodes are stored [k][j][i] with i (the r
 * direction) fastest, so local node l = ((e*p + k)*p + j)*p + i and a field is [E][p][p][p] ("local layout").
 * Element vertex v = a + 2b + 4c sits at (r,s,t) = (2a-1, 2b-1, 2c-1).  nL = E*p^3 must be < 2^31.
 *
 * Memory: every pointer is tagged HOST or DEVICE below.  DEVICE pointers are plain CUDA device pointers (the Python
 * binding passes torch tensors' data_ptr()); they stay owned by the caller and must stay valid until the stream work
 * queued by the call has run.  The context owns the geometric factors, the gather-scatter maps and the PCG work
 * vectors and frees them in sem_ctx_destroy.
 *
 * Execution: sem_ax / sem_gs / sem_ax_gs only enqueue kernels on the context's stream and return (asynchronous).
 * sem_mesh_setup, sem_geom, sem_pcg and the accessors synchronise that stream before returning.
 *
 * Errors: every call returns SEM_OK (0) or a negative code; nothing throws or aborts across the ABI.  There is no
 * CPU fallback: without a CUDA device every compute call returns SEM_ECUDA.
 */
#ifndef SEM_H_
#define SEM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define SEM_API __attribute__((visibility("default")))
#else
#define SEM_API
#endif

typedef struct sem_ctx sem_ctx; /* opaque, library-owned */

typedef enum { SEM_F64 = 0, SEM_F32 = 1 } sem_prec;
typedef enum { SEM_OP_ADD = 0 } sem_op; /* only "exchange-and-sum" is defined by the paper */
typedef enum { SEM_G_STORED = 0, SEM_G_RECOMPUTE = 1 } sem_gmode;

enum {
    SEM_OK = 0,
    SEM_EINVAL = -1, /* bad argument (N<1 or N>15, E<=0, NULL pointer, negative gid, nL>=2^31, bad enum) */
    SEM_EMESH = -2,  /* some Jacobian determinant <= 0 */
    SEM_ECUDA = -3,  /* CUDA runtime error (text in sem_last_error) or no device */
    SEM_ENOMEM = -4, /* device or host allocation failed */
    SEM_ESTATE = -5  /* call order: sem_ax before sem_geom, recompute mode without vertices, ... */
};

/* a0 + a1 (setup).  Builds the context: GLL points/weights/differentiation matrix D for order N (O1)
 * and the canonical gather-scatter maps from one global id per local node ("the user simply provides a
 * global ID for each vertex"; O6):  uniq_gid = distinct gids ascending, l2u[l] = rank of gid[l], mult[g] = copies,
 * seg_off = exclusive scan of mult, seg_idx = local indices stably sorted by gid.
 *   out         HOST   receives the context (NULL on failure, except that a context carrying the error text is
 *                      still returned when the failure happened after allocation; always sem_ctx_destroy it)
 *   vertex_xyz  HOST   [E][8][3] doubles, element vertices (S4/S5: elements are trilinear images of 8 vertices)
 *   gid         HOST or DEVICE (detected) [E][p][p][p] int64, all >= 0 (S11)
 *   dirichlet   HOST, nullable, [E][p^3] bytes, 1 = masked (Dirichlet) node; a unique node is masked if any of its
 *               copies is flagged (S14)
 *   cuda_stream a cudaStream_t (0 = legacy default stream) on which all later work of this context is enqueued */
SEM_API int sem_mesh_setup(sem_ctx** out, int64_t E, int N, const double* vertex_xyz, const int64_t* gid,
                   const uint8_t* dirichlet, void* cuda_stream);

/* a2 (setup).  Geometric factors (P:69 isoparametric map; O3): at every node the Jacobian Jm = dx/dr, detJ, and
 *   G_bc = rho_i rho_j rho_k detJ sum_a (dr_b/dx_a)(dr_c/dx_a), stored (rr,rs,rt,ss,st,tt);  B = rho_i rho_j rho_k detJ.
 *   node_xyz  HOST, nullable, [E][p^3][3]: if given, Jm = D applied to these coordinates (isoparametric); if NULL,
 *             Jm is the analytic derivative of the trilinear blend of the 8 vertices (S5).
 *   mode      SEM_G_STORED: G kept in HBM (48 B/node FP64).  SEM_G_RECOMPUTE: sem_ax recomputes G from the 8
 *             vertices inside the kernel (a9; needs node_xyz == NULL) and no stored G is kept (it is rebuilt for the
 *             duration of sem_get_geom and of the Jacobi-diagonal build).  The operator then moves 16 B per node
 *             instead of 64 and is bound by the FP64 pipe; at N = 7 in FP64 (tensor-core kernel) it is faster than the
 *             stored-G operator once u and w no longer fit in L2 (1.26x at 64^3 elements), slower below; at other
 *             orders the stored-G operator is faster.
 *   with_mass keep B (needed for lambda != 0 and for sem_get_geom's 7th factor)
 * Returns SEM_EMESH if any detJ <= 0.  Also builds the exact assembled diagonal for Jacobi (O7). */
SEM_API int sem_geom(sem_ctx* ctx, const double* node_xyz, sem_gmode mode, int with_mass);

/* a3-a5.  Local operator, no gather-scatter (P:93 contraction; O4):  w = D^T G D u + lambda B u  element by element.
 *   u, w   DEVICE, local layout, nL values of `prec` (double or float); must not alias
 *   lambda Helmholtz shift (S18); lambda != 0 requires with_mass
 * FP32 (S16): u, w, G, D and all accumulation in float (G, D rounded once from double). */
SEM_API int sem_ax(sem_ctx* ctx, const void* u, void* w, sem_prec prec, double lambda);

/* a6.  Gather-scatter QQ^T in place ("exchange-and-sum of shared interface values"; O5): every copy of a
 * unique node receives the sum over all its copies.  No mask is applied.  w DEVICE, local layout. */
SEM_API int sem_gs(sem_ctx* ctx, void* w, sem_prec prec, sem_op op);

/* NEXT-4, first piece: the gather-scatter of several fields in one pass (the paper's `gatherScatterMany`
 * kernel, Table 3; the three velocity components of the Helmholtz solves).  Field f is the local-layout
 * vector at w + f * field_stride (in values of `prec`, field_stride >= nL); every field receives exactly what sem_gs
 * would give it (bit-identical), but the gather-scatter records are read once for up to 4 fields and the value loads of
 * all of them are in flight together.  No mask is applied.  w DEVICE.  Asynchronous on the context's stream.
 * SEM_EINVAL for nfields < 1 or field_stride < nL.
 * field_stride = SEM_INTERLEAVED selects the NODE-INTERLEAVED layout instead: value of field f at local node l is
 * w[l * nfields + f] (2 <= nfields <= 4): the copies of a node then share their 32-byte sectors between the fields,
 * which is what the scattered accesses of the gather-scatter pay for. */
#define SEM_INTERLEAVED 1
SEM_API int sem_gs_many(sem_ctx* ctx, void* w, int nfields, int64_t field_stride, sem_prec prec, sem_op op);

/* NEXT-4: the operator and the Jacobi-PCG solve on several fields that share the geometry ("Each
 * Stokes substep requires the solution of 3 Helmholtz problems -- one for each velocity component -- ... efficiently
 * treated by using Jacobi-preconditioned conjugate gradient iteration").  Field f is the local-layout vector at
 * u + f * field_stride / w + f * field_stride (values of `prec`; field_stride >= nL, even for the FP64 fused path).
 * sem_ax_gs_many: w_f = M QQ^T (D^T G D + lambda B) u_f for every field; each result is what sem_ax_gs gives for that
 *   field (same arithmetic; FP64 p = 8 with stored G: groups of 3 or 2 fields share ONE pass over G, 48 + 16 nf bytes per
 *   node instead of 64 nf; other orders and FP32 run field by field), followed by sem_gs_many's kernels with the mask.
 *   Asynchronous.
 * sem_pcg_many: nfields <= 8 independent Jacobi-PCG solves in lockstep, each with its own alpha, beta, stopping test
 *   (||r_f|| <= tol ||r_f,0||) and breakdown handling, i.e. each field's iterates are those of sem_pcg on it alone; the
 *   operator pass is shared as above.  b, x DEVICE FP64 as in sem_pcg, at field_stride; iters_out, relres_out HOST
 *   [nfields].  On a non-default stream 16 lockstep iterations are one CUDA graph, replayed (as in sem_pcg): three
 *   Helmholtz fields at config 2 take 275 - 281 us per iteration against 3 x 103 us for three sem_pcg solves (the vector
 *   kernels run on groups of 3 or 2 fields and read the Jacobi diagonal and the dot weights once per group).  Synchronises. */
SEM_API int sem_ax_gs_many(sem_ctx* ctx, const void* u, void* w, int nfields, int64_t field_stride, sem_prec prec,
                           double lambda);
SEM_API int sem_pcg_many(sem_ctx* ctx, const double* b, double* x, int nfields, int64_t field_stride, double tol, int maxit,
                         int* iters_out, double* relres_out);

/* NEXT-4: the device side of the gather-scatter across ranks when the elements are partitioned over
 * several GPUs, one context per rank over its own elements with the GLOBAL node ids ("exchange-and-sum of shared
 * interface values").  After the rank-local sem_ax_gs, for every rank r that shares nodes with this one:
 *   sem_iface_pack  buf[q] = w[first local copy of unique node uniq[q]]   (the rank-local sum), q < n
 *   (exchange of the buffers: NCCL send/recv or peer copies, done by the caller -- paper_2110_01716_b200/sharded.py)
 *   sem_iface_add   w[every local copy of unique node uniq[q]] += buf[q];  Dirichlet nodes stay zero
 * with the received buffers added in ascending rank order on every rank.  uniq DEVICE int32 [n]: rank-local unique-node
 * indices (positions in sem_get_maps' uniq_gid) of the shared nodes, in ascending global id -- the same order on both
 * sides; each node at most once per list.  buf, w DEVICE, `prec` values.  Asynchronous on the context's stream. */
SEM_API int sem_iface_pack(sem_ctx* ctx, const int32_t* uniq, int64_t n, const void* w, void* buf, sem_prec prec);
SEM_API int sem_iface_add(sem_ctx* ctx, const int32_t* uniq, int64_t n, const void* buf, void* w, sem_prec prec);

/* NEXT-4, the sharded operator and solver (P:89 overlap of the non-local gather-scatter with interior work; P:101;
 * P:119-121).  The library runs every kernel; the transport between ranks is the caller's and reaches the library
 * through three hooks, each called on the host from inside the library call and expected to ORDER its work on the
 * context's stream (enqueue and return; no host synchronisation needed) and to return 0 on success:
 *   gs_begin(user, w, prec)    the rank-local sums of all nodes shared with other ranks are final in w (DEVICE, [nL]
 *                              values of sem_prec `prec`): pack them (sem_iface_pack) and start sending/receiving;
 *   gs_end(user, w, prec)      wait for the peers' buffers and add them (sem_iface_add, ascending rank order);
 *                              between the two calls the library launches work that touches no shared node;
 *   allreduce(user, s, n)      s DEVICE double[n]: replace by the sum over all ranks, the same bits on every rank.
 * The hooks struct is read during the call only.  Dirichlet flags must agree between the ranks on shared nodes. */
typedef struct sem_shard_hooks {
    int (*gs_begin)(void* user, void* w, int prec);
    int (*gs_end)(void* user, void* w, int prec);
    int (*allreduce)(void* user, double* scalars, int n);
    void* user;
} sem_shard_hooks;

/* Declares that elements [0, n_iface_elems) of this context are the only ones that touch nodes shared with other ranks
 * (the caller orders its elements that way; 0 = unknown, no overlap).  The sharded calls then run operator and
 * gather-scatter of those elements first, call gs_begin, run the remaining elements, and call gs_end: the exchange
 * overlaps the interior work (A18).  Rounded up to whole element groups.  Drops cached graphs.  Host call. */
SEM_API int sem_shard_set_interface(sem_ctx* ctx, int64_t n_iface_elems);

/* The chunks sem_ax_gs / sem_pcg work in (fields larger than L2, or the interface split): *n_chunks (1 = one launch
 * pair), their element bounds (HOST, n_chunks + 1 values, cap = room in elem_bounds; NULL to skip) and how many leading
 * chunks precede gs_begin in the sharded calls (0 = none).  Any pointer may be NULL.  Host call. */
SEM_API int sem_get_chunks(sem_ctx* ctx, int64_t* elem_bounds, int cap, int* n_chunks, int* iface_chunks);

/* w = M QQ^T (D^T G D + lambda B) u with QQ^T summing over ALL ranks' copies: sem_ax_gs on this rank's elements with the
 * exchange through the hooks.  Same arguments as sem_ax_gs.  Nodes that live on one rank only are bit-identical to
 * the single-context result when their copies are summed in the same order (always for 1 or 2 copies; for more when
 * the rank keeps the caller's element order); everything else agrees to round-off. */
SEM_API int sem_ax_gs_sharded(sem_ctx* ctx, const void* u, void* w, sem_prec prec, double lambda,
                              const sem_shard_hooks* hooks);

/* a8 on the partitioned mesh: every rank calls this with its part of b and x (DEVICE, [nL] of its context, x 16-byte
 * aligned) and the same tol / maxit.  The recurrence, stopping test and breakdown rule are sem_pcg's (S12-S14); the
 * dots are summed over ranks by TWO all-reduces per iteration (p.q; r.r and r.z together), in place on device scalars,
 * so every rank takes the same decisions; the Jacobi diagonal and the dot weights (1 / multiplicity) are assembled over
 * all ranks through the hooks at the first call and when lambda changes.  iters_out / relres_out / the history
 * (sem_get_pcg_history) are the same on every rank.  Synchronises the stream every 8 iterations. */
SEM_API int sem_pcg_sharded(sem_ctx* ctx, const double* b, double* x, double tol, int maxit,
                            const sem_shard_hooks* hooks, int* iters_out, double* relres_out);

/* a3-a7.  w = M QQ^T (D^T G D + lambda B) u, with M zeroing Dirichlet nodes (if the context has any).  u must be
 * continuous (equal on all copies of a shared node).  Called repeatedly with the same (u, w, prec, lambda) on a
 * non-default stream, the second call records the two kernels into a CUDA graph and later calls replay it (still
 * asynchronous; the graph is dropped when the arguments, the geometry or the variant change). */
SEM_API int sem_ax_gs(sem_ctx* ctx, const void* u, void* w, sem_prec prec, double lambda);

/* a8.  Jacobi-preconditioned conjugate gradients on M QQ^T A_L M (O8, S12-S14), FP64, lambda = 0 unless
 * set with sem_set_lambda:
 *   x = M x0; r = M b - A x (b if x0 == 0); z = Minv r; p = z; rho = r.z; r0 = ||r||
 *   repeat: q = A p; alpha = rho / p.q; x += alpha p; r -= alpha q; stop if ||r|| <= tol r0 or it == maxit;
 *           z = Minv r; beta = r.z / rho; p = z + beta p
 * with dots over unique unmasked nodes.  b (assembled right-hand side) and x are DEVICE, local layout, continuous.
 *   iters_out   HOST  number of operator applications in the loop
 *   relres_out  HOST  ||r|| / r0 from the recurrence
 * Reaching maxit is not an error; r0 == 0 (e.g. b == 0 with x0 == 0) returns x = M x0 after 0 iterations;
 * p.q <= 0 stops (breakdown) with SEM_OK.
 * Execution: all scalars stay on the device (no host round trip per iteration; the host polls a flag every 16
 * iterations); on a non-default stream 16 iterations are one CUDA graph, replayed.  The dot products are reduced with
 * FP64 atomics, so iterates are repeatable to round-off, not bit for bit.  On a large mesh (fields > 256 MB) whose
 * element order has no locality the loop runs on an inner copy of the context with the elements sorted by smallest
 * global id (b and x are gathered / scattered in element blocks); results are unchanged to round-off. */
SEM_API int sem_pcg(sem_ctx* ctx, const double* b, double* x, double tol, int maxit, int* iters_out, double* relres_out);

/* Helmholtz shift used by sem_pcg and by the Jacobi diagonal (default 0).  Requires with_mass if != 0. */
SEM_API int sem_set_lambda(sem_ctx* ctx, double lambda);

/* Residual history of the last sem_pcg: hist[i] = ||r_i|| / r0 for i = 0..min(iters, n-1).  hist HOST. */
SEM_API int sem_get_pcg_history(sem_ctx* ctx, double* hist, int n);

/* Parity accessors: copy library-owned data to caller-provided HOST buffers (any may be NULL = skip). */
SEM_API int sem_get_counts(sem_ctx* ctx, int64_t* nL, int64_t* U, int64_t* S, int64_t* Us);
SEM_API int sem_get_maps(sem_ctx* ctx, int32_t* l2u /*[nL]*/, int32_t* mult /*[U]*/, int64_t* seg_off /*[U+1]*/,
                 int32_t* seg_idx /*[nL]*/, int64_t* uniq_gid /*[U]*/);
SEM_API int sem_get_gll(sem_ctx* ctx, double* xi /*[p]*/, double* rho /*[p]*/, double* D /*[p][p] row = point*/);
SEM_API int sem_get_geom(sem_ctx* ctx, double* G /*[E][6 or 7][p^3]*/, double* detJ /*[E][p^3]*/);
SEM_API int sem_get_diag(sem_ctx* ctx, double* diagA_local /* assembled QQ^T diag(A_L), unmasked, [E][p^3] */);

/* NEXT-1.  p-multigrid transfer between two discretisations of the SAME E elements ("u_f =
 * (J x J x J) u_c, where J is the 1D polynomial interpolation operator from the coarse GLL points to the fine GLL
 * points"), element by element, no gather-scatter and no weighting (the multigrid cycle applies those):
 *   SEM_PROLONG:   out[E][pf^3] = (J   x J   x J  ) in[E][pc^3]
 *   SEM_RESTRICT:  out[E][pc^3] = (J^T x J^T x J^T) in[E][pf^3]
 * J[i][j] = Lagrange cardinal function j of the coarse GLL points at fine GLL point i ([pf][pc], pc = N_c+1 <= pf).
 *   coarse, fine  contexts from sem_mesh_setup with equal E and N_c <= N_f (else SEM_EINVAL, text in fine's error)
 *   in, out       DEVICE, local layout, `prec` values; must not alias
 * Asynchronous on the FINE context's stream.  FP32 (S16): J rounded once from double, accumulation in float. */
typedef enum { SEM_PROLONG = 0, SEM_RESTRICT = 1 } sem_transfer_dir;
SEM_API int sem_transfer(sem_ctx* coarse, sem_ctx* fine, const void* in, void* out, sem_prec prec, sem_transfer_dir dir);
/* Parity accessor: the interpolation matrix J, [pf][pc] doubles, HOST. */
SEM_API int sem_get_interp(sem_ctx* coarse, sem_ctx* fine, double* J);

/* NEXT-1.  Chebyshev-accelerated point-Jacobi smoother, `order` steps on
 * M QQ^T (D^T G D + lambda B) M with the exact Jacobi diagonal (O7), for eigenvalue bounds [lmin, lmax] of diag^-1 A
 * given by the caller (reading S23 in DESIGN.md; the recurrence is written out in csrc/sem_cheby.cu):
 *   x <- x + p(diag^-1 A) diag^-1 (b - A x),  error multiplied by T_order((theta - t)/delta) / T_order(theta/delta)
 *   b, x        DEVICE, local layout, continuous, `prec` values; b assembled; x: in = initial guess (masked on entry),
 *               out = smoothed iterate; must not alias; x 16-byte aligned
 *   zero_guess  != 0: x is taken as 0 and not read (saves one operator application)
 * `order` operator applications (order - 1 with zero_guess).  Asynchronous on the context's stream.
 * SEM_EINVAL for order < 1 or bounds not 0 < lmin < lmax. */
SEM_API int sem_cheby(sem_ctx* ctx, const void* b, void* x, int order, double lmin, double lmax, int zero_guess,
                      sem_prec prec);

/* Setup helper for the bounds above: `iters` power iterations on diag^-1 A (FP64, synchronises); *lam_out is the last
 * estimate ||diag^-1 A v|| / ||v||, which approaches lambda_max from below: multiply by a safety factor (1.1). */
SEM_API int sem_lambda_max(sem_ctx* ctx, int iters, double* lam_out);

/* The Chebyshev-Jacobi smoother of sem_cheby, FP64, for callers that cannot allocate device memory (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc).  It calls no cudaMalloc / cudaFree and no allocating
 * library routine: its three work vectors live in a static device array inside the library, 3 x SEM_NOALLOC_MAX_NODES
 * doubles (12 MB, held by every GPU that loads the library until the process exits).  b, x, order, lmin, lmax,
 * zero_guess as in sem_cheby; the result equals sem_cheby's matrix-free FP64 path.
 * Requirements: nL <= SEM_NOALLOC_MAX_NODES (else SEM_EINVAL with a message naming the limit); stored geometric
 * factors; the Jacobi diagonal already built for the current lambda by an earlier sem_get_diag / sem_cheby / sem_pcg
 * call (else SEM_ESTATE: building it would allocate); the context's device current.  The first call on a device
 * resolves the array's address (cudaGetSymbolAddress; no allocation) -- make it outside stream capture.
 * Every call on a device, from any context, shares the array, which keeps the previous call's contents (a call only
 * reads what it wrote itself, nothing needs clearing): calls that overlap on the GPU (different streams) race.
 * Asynchronous on the context's stream. */
#define SEM_NOALLOC_MAX_NODES (1 << 19)
SEM_API int sem_cheby_noalloc(sem_ctx* ctx, const double* b, double* x, int order, double lmin, double lmax,
                              int zero_guess);

/* NEXT-1c.  p-multigrid V-cycle preconditioner z = M^-1 r over `nlevels` contexts, finest first
 * (the cycle is reading S25 in DESIGN.md and is written out in csrc/sem_pmg.cu): Chebyshev-Jacobi
 * pre- and post-smoothing of `smooth_order` steps on every level but the coarsest, multiplicity-weighted restriction
 * J^T, prolongation J, `coarse_order` Chebyshev-Jacobi steps on the coarsest level.
 *   levels      HOST array of contexts after sem_geom: equal E, strictly decreasing N, the same stream, all with or
 *               all without a Dirichlet mask.  They must outlive the sem_pmg.
 *   lmin, lmax  HOST [nlevels], eigenvalue bounds of diag^-1 A per level (S23)
 *   prec        precision of r, z and of every step of the cycle (the paper runs it in FP32)
 * sem_pmg_vcycle: r, z DEVICE, finest level's local layout, continuous, r assembled; z is overwritten; 16-byte aligned;
 * asynchronous on the levels' stream.  The sem_pmg owns its work vectors; sem_pmg_destroy frees them. */
typedef struct sem_pmg sem_pmg;
SEM_API int sem_pmg_create(sem_pmg** out, int nlevels, sem_ctx* const* levels, const double* lmin, const double* lmax,
                           int smooth_order, int coarse_order, sem_prec prec);
SEM_API int sem_pmg_vcycle(sem_pmg* mg, const void* r, void* z);
SEM_API void sem_pmg_destroy(sem_pmg* mg);
/* Flexible PCG on the finest level of `mg` with the V-cycle as preconditioner (reading S26): the recurrence of sem_pcg
 * with the Polak-Ribiere beta = r_new.(z_new - z_old) / (r_old.z_old), FP64 outer iteration, x0 = 0, the cycle in mg's
 * precision.  b, x DEVICE FP64, finest local layout, continuous, b assembled; x is overwritten.  Synchronises.
 * iters_out / relres_out as in sem_pcg; sem_pmg_get_history copies ||r_k||/||r_0||, k = 0..min(iters, n-1), to HOST. */
SEM_API int sem_fpcg(sem_pmg* mg, const double* b, double* x, double tol, int maxit, int* iters_out, double* relres_out);
SEM_API int sem_pmg_get_history(sem_pmg* mg, double* hist, int n);

/* NEXT-3.  Projection onto previous solutions (reading S27 in DESIGN.md): an A-orthonormal
 * basis P_L of up to Lmax earlier solution updates, A = the context's masked assembled operator (current lambda).
 *   sem_proj_guess   xbar = P_L P_L^T b (the A-norm best fit in span P_L; 0 while the space is empty) and
 *                    b_reduced = b - A xbar, the right-hand side of the reduced problem A dx = b_reduced.  Asynchronous.
 *   sem_proj_update  after the caller has solved the reduced problem: dx is A-orthonormalised against P_L (one round of
 *                    classical Gram-Schmidt, one reduction) and appended; the space restarts (is emptied first) when it
 *                    already holds Lmax vectors; *accepted = 0 if dx was (numerically) inside the space.  One operator
 *                    application; synchronises.
 * b, xbar, b_reduced, dx: DEVICE, FP64, local layout, continuous; b assembled; dx 16-byte aligned.  The context must
 * outlive the sem_proj, which owns 2 Lmax + 1 vectors of device memory. */
typedef struct sem_proj sem_proj;
SEM_API int sem_proj_create(sem_proj** out, sem_ctx* ctx, int Lmax);
SEM_API int sem_proj_guess(sem_proj* pj, const double* b, double* xbar, double* b_reduced);
SEM_API int sem_proj_update(sem_proj* pj, const double* dx, int* accepted);
SEM_API int sem_proj_size(sem_proj* pj, int* L);
SEM_API void sem_proj_destroy(sem_proj* pj);

/* NEXT-2a.  Fast-diagonalisation local solve of the Schwarz smoothers, Eq. (3): for every
 * element e of the context
 *      u^e = (S_z x S_y x S_x) Lambda^-1 (S_z^T x S_y^T x S_x^T) b^e
 * on the element's extended m x m x m block (m = N + 3 in the paper: "for an 8 x 8 x 8 brick (N = 7), one solves a
 * 10 x 10 x 10 local problem"; any 2 <= m <= 16 is accepted and m need not be related to the context's N).  With
 * S_d^T B_d S_d = I, S_d^T A_d S_d = diag(lam_d) and Lambda[c][b][a] = lam_x[a] + lam_y[b] + lam_z[c] this is the exact
 * inverse of Bz x By x Ax + Bz x Ay x Bx + Az x By x Bx.  Building the blocks (the face-only exchange of P:107), the
 * weighting and the sum back into the residual are not part of this call (NEXT-2b).
 *   S           DEVICE [E][3][m][m]: direction d = 0,1,2 = x,y,z; S_d[row][col] row-major, eigenvectors in columns
 *   inv_lambda  DEVICE [E][m][m][m]: 1/Lambda, eigen-indices [c][b][a] (z, y, x; x fastest)
 *   b, u        DEVICE [E][m][m][m], [k][j][i] with i (x) fastest; u may alias b (in place)
 * All four arrays hold `prec` values (S and inv_lambda rounded by the caller; accumulation in `prec`) and are 16-byte
 * aligned (SEM_EINVAL otherwise).
 * Asynchronous on the context's stream; needs only sem_mesh_setup (E and the stream).  SEM_EINVAL for m outside 2..16. */
SEM_API int sem_fdm_apply(sem_ctx* ctx, int m, const void* S, const void* inv_lambda, const void* b, void* u,
                          sem_prec prec);

/* NEXT-2a setup (host, synchronous, no context, no device): the eigen-decompositions behind sem_fdm_apply.  For every
 * element and direction d the generalised symmetric eigenproblem A_d s = lambda B_d s is solved with S_d^T B_d S_d = I
 * (Cholesky of B_d + cyclic Jacobi; "fast diagonalization (FDM) Deville et al. (2002)"), and
 * inv_lambda[c][b][a] = 1 / (lambda_x[a] + lambda_y[b] + lambda_z[c]).
 *   A, B        HOST [E][3][m][m] doubles (d = x, y, z), symmetric (the symmetric part is used), B positive definite
 *   S           HOST out [E][3][m][m]: eigenvectors in columns, eigenvalues ascending; a column's sign is arbitrary
 *               (Eq. (3) does not depend on it)
 *   inv_lambda  HOST out [E][m][m][m]
 * Round S and inv_lambda to the precision sem_fdm_apply is called with.  SEM_EINVAL for NULL pointers, E <= 0,
 * m outside 2..16 or a B_d that is not positive definite. */
SEM_API int sem_fdm_setup(int64_t E, int m, const double* A, const double* B, double* S, double* inv_lambda);

/* NEXT-2b.  The overlapping additive Schwarz smoother around sem_fdm_apply ("The Schwarz smoothers
 * are implemented by solving local Poisson problems on domains extended into adjacent elements by one layer"
 * "We exchange face data only to get the domain extensions -- meaning 6 exchanges per element instead of 26", the
 * restricted variant "that does not require communication after the local solve"; Table 2 `gs_ext`, `fdm`, `fdm_apply`).
 * The paper cites Lottes & Fischer (2005) and prints no formula; the construction is reading S29 of DESIGN.md:
 *   block of element e: m = N + 3 points per direction: index 1..N+1 its own nodes, index 0 / m-1 the face neighbour's
 *     node one layer in from the shared face; only the 6 face layers are filled, block edges and corners hold no node;
 *   A~_e = Bz x By x Ax + Bz x Ay x Bx + Az x By x Bx from the 1-D pairs of the line [left | element | right]: the 1-D
 *     spectral-element matrices (2/L) D^T diag(rho) D, (L/2) diag(rho) of the three segments assembled and the m retained
 *     rows/columns kept; L = mean length of the element's 4 edges in that local direction; without a neighbour the ghost
 *     point is a decoupled unit row, on a Dirichlet face the face node too;
 *   z = M W^1/2 QQ^T sum_e R_e^T A~_e^-1 R_e (W^1/2 r),  W = 1 / (block positions mapping to the node), split over both
 *     sides so that S is symmetric positive definite; SEM_SCHWARZ_RAS scatters back the element's own nodes only and
 *     weights the result by W = 1 / multiplicity (not symmetric).
 * sem_schwarz_setup (after sem_geom; N >= 2, else SEM_EINVAL; synchronises; host work O(E)): finds the face neighbours
 * from the gather-scatter maps, builds the 1-D pairs, their eigen-decompositions (as sem_fdm_setup) in FP64 and FP32, and
 * both weight vectors.  sem_geom discards it.  SEM_EMESH if a shared face cannot be matched node for node.
 * sem_schwarz: r, z DEVICE, local layout, continuous, `prec` values, r assembled; z may alias r.  Three element-local
 * kernels (extension gather, Eq. (3) in place, weighted combination) and the gather-scatter with the Dirichlet mask;
 * asynchronous on the context's stream.  SEM_ESTATE before sem_schwarz_setup.
 * sem_get_schwarz (parity accessor, HOST buffers, any may be NULL): nbr [E][6] (face f = 2 axis + side; -1 = boundary),
 * A, B [E][3][m][m] the 1-D pairs, W [E][p^3] the weight vector of `kind` as applied (ASM: W^1/2; RAS: W). */
typedef enum { SEM_SCHWARZ_ASM = 0, SEM_SCHWARZ_RAS = 1 } sem_schwarz_kind;
SEM_API int sem_schwarz_setup(sem_ctx* ctx);
SEM_API int sem_schwarz(sem_ctx* ctx, const void* r, void* z, sem_prec prec, sem_schwarz_kind kind);
SEM_API int sem_get_schwarz(sem_ctx* ctx, int32_t* nbr, double* A, double* B, double* W, sem_schwarz_kind kind);

/* Chebyshev-accelerated Schwarz ("Chebyshev-accelerated overlapping Schwarz"; "we switched from
 * Chebyshev-Jacobi to Chebyshev-Schwarz"): the recurrence of sem_cheby with the Schwarz operator S in place of diag^-1,
 * for bounds [lmin, lmax] of S A given by the caller (sem_lambda_max_schwarz).  Arguments as sem_cheby. */
SEM_API int sem_cheby_schwarz(sem_ctx* ctx, const void* b, void* x, int order, double lmin, double lmax, int zero_guess,
                              sem_prec prec, sem_schwarz_kind kind);
/* `iters` power iterations on S A (FP64, synchronises): the last estimate ||S A v|| / ||v||, as sem_lambda_max. */
SEM_API int sem_lambda_max_schwarz(sem_ctx* ctx, sem_schwarz_kind kind, int iters, double* lam_out);

/* Smoother of a sem_pmg (default SEM_SMOOTH_CHEBY_JACOBI).  With SEM_SMOOTH_CHEBY_SCHWARZ / _RAS every level with N >= 2
 * is smoothed by sem_cheby_schwarz of `smooth_order` steps (sem_schwarz_setup is run on it if needed) with the bounds
 * given here; levels with N = 1 and the coarsest level keep Chebyshev-Jacobi with the bounds of sem_pmg_create.
 *   lmin, lmax  HOST [nlevels], bounds of S A per level (ignored where Jacobi stays).  Drops recorded graphs. */
typedef enum { SEM_SMOOTH_CHEBY_JACOBI = 0, SEM_SMOOTH_CHEBY_SCHWARZ = 1, SEM_SMOOTH_CHEBY_RAS = 2 } sem_smoother;
SEM_API int sem_pmg_set_smoother(sem_pmg* mg, sem_smoother smoother, const double* lmin, const double* lmax);

/* Measurement helper ("FP64 peak ... measure it"): a register-resident arithmetic microbenchmark on
 * the current device, best of 5 launches after one warm-up, CUDA-event timed on `cuda_stream`; synchronises.  Not part
 * of the method: bench.py quotes the FP64-ALU-bound kernels (a9 recomputed G, the fast-diagonalisation solve) against it.
 *   kind        SEM_PEAK_FMA_F64 / SEM_PEAK_FMA_F32: independent FMA chains;  SEM_PEAK_DMMA_F64: mma.sync m8n8k4 f64
 *   tflops_out  HOST  2 flops per FMA
 * SEM_EINVAL for a bad kind or NULL; SEM_ECUDA without a device. */
enum { SEM_PEAK_FMA_F64 = 0, SEM_PEAK_FMA_F32 = 1, SEM_PEAK_DMMA_F64 = 2 };
SEM_API int sem_measure_peak(int kind, void* cuda_stream, double* tflops_out);

/* Tuning knob for experiments: selects the Ax kernel variant.  0 = the default per (precision, p): p = 8 runs on the
 * tensor cores, one warp per element (FP64: r/s contractions as DMMA m8n8k4; FP32: as TF32 m16n8k8 in three passes,
 * FP32-level accuracy), every other p <= 12 the streaming kernel; 1 = the simple plain-load kernel; 2 = the scalar
 * streaming kernel (p <= 12); 3 = FP64 p = 8 only: the DMMA kernel with 5 ring stages and 8 warps per SM; 4 = the
 * pencil kernel (8 <= p <= 12: every 1-D contraction by a thread that owns a whole line of p values; the default for
 * FP32 p = 9 and FP64 p = 12, where it measured faster than the streaming kernel).
 * 100 + v selects the kernel of sem_fdm_apply / the fused restricted Schwarz instead: 100 = the scalar line kernels
 * (default), 101 = FP32, 6 <= m <= 12: the tensor-core kernel (every 1-D contraction as TF32 m16n8k8 in three passes;
 * measured slower than the scalar kernels at every m, kept as the measurement north_star asks for).
 * Environment knobs read at setup (tests, experiments): SEM_CHUNK_GROUPS = element groups per chunk of the chunked
 * operator / gather-scatter (fields larger than L2; a huge value disables it); SEM_INNER = 0 / 1 never / always build the
 * renumbered inner context that sem_pcg uses on large meshes without locality; SEM_COARSE = 0 keeps sem_cheby at N = 1
 * on the matrix-free operator (default: the assembled N = 1 operator, one kernel per Chebyshev step). */
SEM_API int sem_set_variant(sem_ctx* ctx, int ax_variant);

/* Last error text of this context ("" if none); valid until the next call on the context.  NULL ctx -> static text. */
SEM_API const char* sem_last_error(sem_ctx* ctx);

SEM_API void sem_ctx_destroy(sem_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* SEM_H_ */
