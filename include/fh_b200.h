/*
 * fh_b200.h -- C ABI of the B200-native hot path of U(1)xSU(2)-symmetric two-site TDVP for
 * the 1D Fermi-Hubbard chain (arxiv/paper_2606_04771; citations are PAPER.md:<line>).
 *
 * Every function returns int: 0 = FH_OK, negative = FH_E* code; fh_last_error(ctx) returns a
 * NUL-terminated message owned by the library (valid until the next failing call on ctx).
 * A context is not thread-safe.  All device work is enqueued on the cudaStream_t given at
 * context creation; calls that return host data synchronise that stream before returning.
 *
 * Conventions (readings A-1, F-2, F-4):
 *   sector label (q, tj): q = N_up - N_dn (integer), tj = 2*T (doubled pseudospin)  -- the
 *     U(1)_spin x SU(2)_charge symmetry of PAPER.md:41, 208; bond spaces decompose as Eq. (7)
 *     PAPER.md:210-214 with degeneracy d_{q,tj};
 *   site multiplets s: 0 = (+1,0) |up>, 1 = (-1,0) |dn>, 2 = (0,1/2) {|0>, eps_i |updn>};
 *   MPO bond multiplets w: 0 = S (0,0), 1 = P (+1,1/2), 2 = M (-1,1/2), 3 = F (0,0)  (W = 4,
 *     PAPER.md:260);
 *   a block is a dense row-major complex128 matrix (interleaved re,im; 16 B per element):
 *     site tensor   A[a,s,c]            d_a  x d_c
 *     two-site      theta[a,s1,c,s2,b]  d_a  x d_b   (c = intermediate coupling label)
 *     environments  L[a',w,a]           d_a' x d_a ,  R[b',w,b]  d_b' x d_b
 *   blocks of one tensor are stored contiguously in the canonical (lexicographic, sectors
 *   ordered by (q, tj)) order of their label tuples; "planned block order" below means that.
 *   (The vectors heff_apply works on have a layout of their own: see heff_import / heff_export.)
 *
 * Pointer arguments are HOST pointers unless the name ends in _dev.
 */
#ifndef FH_B200_H
#define FH_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FH_OK 0
#define FH_EINVAL (-1)   /* bad argument (odd L, unknown label, size mismatch, ...) */
#define FH_ENOMEM (-2)   /* arena exhausted */
#define FH_ECUDA (-3)    /* CUDA / cuSOLVER runtime error */
#define FH_ESTATE (-4)   /* call out of order (e.g. heff_apply without heff_plan) */

typedef struct fh_ctx fh_ctx;
typedef struct fh_mpo fh_mpo;
typedef struct fh_mps fh_mps;

/* ---- context ---------------------------------------------------------------------------
 * cuda_stream: a cudaStream_t (NULL = legacy default stream).  arena_dev: device pointer to
 * arena_bytes bytes owned by the caller (e.g. a torch tensor) that must outlive the context,
 * or NULL, in which case the library cudaMalloc()s arena_bytes and frees them on destroy.
 * All tensors (MPS, environments, Krylov vectors, scratch) live in this one HBM arena. */
int fh_ctx_create(fh_ctx** out, void* cuda_stream, void* arena_dev, size_t arena_bytes);
void fh_ctx_destroy(fh_ctx* ctx);
/* message of the last failing call on ctx; with ctx = NULL: why the last fh_ctx_create of this thread failed */
const char* fh_last_error(const fh_ctx* ctx);
/* Options of a context (host-only; FH_EINVAL on a NULL context, an unknown key or a value out of range).
 *   FH_OPT_GEMM_PATH     which form of the grouped ZGEMM heff_apply uses for two-site plans: 0 = the library
 *                        chooses by the size of the plan (default), 1 = one warp-unit per one-warp CTA, two
 *                        launches (csrc/zgemm.cu), 2 = warp-specialised persistent kernel, both stages in one
 *                        launch (csrc/zgemm_ws.cu), 3 = the warp units of form 1 with both stages in ONE launch
 *                        (stage-2 units wait on per-output counters; set it before heff_plan; bit-identical to
 *                        form 1).  Same results to rounding (the k-split tiles of form 2 add partial sums in
 *                        another, fixed, order).
 *   FH_OPT_SVD_MID_MAXN  widest sector matrix (columns) the library's own global-memory Jacobi kernel takes
 *                        instead of the vendor SVD, 0 .. 256 (default 100; 0 = none).
 *   FH_OPT_SVD_THREADS   host threads that drive the vendor SVD / QR routines, 1 .. 12 (default: cores - 1,
 *                        at most 12); takes effect before the first factorisation of the context.
 *   FH_OPT_SVD_SMALL_MAXN widest sector matrix (columns) the shared-memory Jacobi / Householder kernels take, provided
 *                        it fits their shared memory, 0 .. 4096 (default 4096 = whatever fits; 0 = none: every
 *                        matrix goes to the next route).  With FH_OPT_SVD_MID_MAXN this lets a test send small
 *                        matrices through every factorisation route. */
#define FH_OPT_GEMM_PATH 1
#define FH_OPT_SVD_MID_MAXN 2
#define FH_OPT_SVD_THREADS 3
#define FH_OPT_SVD_SMALL_MAXN 4
/*   FH_OPT_SYMMETRY      label algebra of every object created in the context afterwards: 0 =
 *                        U(1)_spin x SU(2)_charge (default; the conventions at the top of this header), 1 = U(1) x U(1)
 *                        (PAPER.md:59, 66, 296): labels (q, 0) with q = (N_up - N_dn) + 64 (N - k) on bond k, site
 *                        states s = 0 |0>, 1 |up>, 2 |dn>, 3 |updn>; MPO bond states 0 = I, 1 = c+_up P, 2 = c+_dn P,
 *                        3 = c_up P, 4 = c_dn P, 5 = final (W = 6), all recoupling coefficients 1, MPO of Eq. (1) as it
 *                        stands.  Set it before fh_mpo_build / mps_create and do not change it while they live. */
#define FH_OPT_SYMMETRY 5
/*   FH_OPT_PRECISION     arithmetic of the two-site heff_apply (and of every Lanczos step of tdvp2_sweep / heff_expm
 *                        on a two-site plan): 0 = complex128 on the FP64 tensor pipe (default), 1 = split precision
 *                        (PAPER.md:264-270): operands, intermediate and result stay complex128 in
 *                        memory, every product is taken as 3 x TF32 (x = hi + lo, a b ~ hi hi + hi lo + lo hi) on the
 *                        tcgen05 tensor cores with float32 accumulation in tensor memory: single-precision class
 *                        error (<= ~1e-6 relative Frobenius per apply; oracle/splitprec.py states the bounds).
 *                        One-site applies, environment updates, vector kernels and the SVD stay FP64. */
#define FH_OPT_PRECISION 6
/*   FH_OPT_SVD_GRAM_MINN narrowest sector matrix (columns, 0 .. 65536; default 104; 0 = never) among those the vendor
 *                        SVD would take that is factorised through its Gram matrix instead: G = B^H B, Hermitian
 *                        eigendecomposition (cusolverDnZheevd), U = B V / sigma.  2.7 x faster per matrix at 600
 *                        columns, and the largest sector matrix of a bond is the critical path of the SVD phase.
 *                        Accurate for the singular values a chi-capped truncation keeps (error eps sigma_max^2 /
 *                        sigma_i); a sector whose smallest KEPT singular value is below 3e-3 of its largest is redone
 *                        by the vendor SVD before the bond is updated (fh_factorization_stats [7], [8]). */
#define FH_OPT_SVD_GRAM_MINN 7
/*   FH_OPT_SVD_GRAM_BATCH_MAXN widest Gram-route sector matrix (columns; default 256; 0 = none) whose eigenproblem is
 *                        solved together with those of the other such sectors of the bond in ONE batched vendor call
 *                        (cusolverDnXsyevBatched on Gram matrices padded to a common size) instead of one call per
 *                        matrix: the vendor eigensolvers are chains of small dependent kernels and a bond's sixteen
 *                        chains queue on the GPU front end; the batched solver walks one chain for all of them. */
#define FH_OPT_SVD_GRAM_BATCH_MAXN 8
int fh_set_option(fh_ctx* ctx, int key, int value);
/* bytes currently allocated / high-water mark in the arena */
int fh_arena_stats(const fh_ctx* ctx, size_t* used_bytes, size_t* peak_bytes);

/* ---- model: Eq. (1) PAPER.md:26-30 -----------------------------------------------------
 * Builds the reduced MPO (bond multiplets S,P,M,F) of H_sym = hopping + (U/2) sum_i P_D,i,
 * which equals Eq. (1) on the half-filled sector (reading A-2).  L even, 2 <= L <= 4096. */
int fh_mpo_build(fh_ctx* ctx, int L, double t_h, double U, fh_mpo** out);
void fh_mpo_destroy(fh_mpo* mpo);
/* reduced MPO element table of one site: val[6][6][4][4] = W[w][w'][s'][s], rank2[6][6] = doubled
 * operator rank of (w,w') or -1 when the pair is absent (the SU(2) mode uses w < 4, s < 3). */
int fh_mpo_get_site(const fh_mpo* mpo, int site, double* val, int32_t* rank2);

/* ---- state -----------------------------------------------------------------------------
 * mps_init_neel: Eq. (2), |up,dn,up,dn,...>, one 1x1 block per site, every bond
 * a single sector with d = 1; orthogonality centre at site 0; environments R_1..R_L built. */
int mps_init_neel(fh_ctx* ctx, const fh_mpo* mpo, int L, fh_mps** out);
/* empty MPS of L sites for synthetic workloads (BASELINE.json configs 2-5) */
int mps_create(fh_ctx* ctx, int L, fh_mps** out);
void mps_destroy(fh_ctx* ctx, fh_mps* mps);
/* Sector table of bond k (k sites to its left), k = 0..L: n labels, sorted by (q,tj). */
int mps_set_bond(fh_ctx* ctx, fh_mps* mps, int bond, int n, const int32_t* q, const int32_t* tj,
                 const int32_t* d);
int mps_get_bond(const fh_mps* mps, int bond, int* n, int32_t* q, int32_t* tj, int32_t* d);
/* Number of blocks / total complex elements of site tensor `site` given its two bond tables
 * (all fusion-allowed (a,s,c)), and the labels[nblk][5] = (qa,tja,s,qc,tjc), dims[nblk][2]. */
int mps_site_layout(const fh_mps* mps, int site, int* nblk, int64_t* nelem, int32_t* labels,
                    int32_t* dims);
/* Upload / download a whole site tensor: `data` holds the blocks back to back in planned block
 * order.  data_is_device != 0: device pointer (copied D2D on the context stream).  The getters take the capacity
 * of `data` in complex128 elements and return FH_EINVAL, copying nothing, when it is below the layout's nelem. */
int mps_set_site(fh_ctx* ctx, fh_mps* mps, int site, const void* data, int data_is_device);
int mps_get_site(fh_ctx* ctx, const fh_mps* mps, int site, void* data, int64_t capacity_elems, int data_is_device);
/* Checkpoint / resume for long runs (the paper's take up to 16 h).  mps_save writes the bond tables
 * and the site tensors of a state whose orthogonality centre is on site 0 (the state every sweep returns) to a
 * binary file (host byte order; header "FHMPS01", L, the tdvp_sweep_auto flag, per bond n x (q, 2j, d), per site
 * the element count and the complex128 blocks in layout order).  mps_load rebuilds the state in this context and
 * recomputes R_1..R_L with the given MPO, so that tdvp2_sweep / tdvp1_sweep / measure_* continue from it.
 * FH_EINVAL: file cannot be opened, is truncated, or does not match the MPO's chain length. */
int mps_save(fh_ctx* ctx, const fh_mps* mps, const char* path);
int mps_load(fh_ctx* ctx, const fh_mpo* mpo, const char* path, fh_mps** out);
/* Release the arena storage of one site tensor (streamed environment construction at large chi,
 * BASELINE.json config 5: a site is uploaded, absorbed into an environment, then dropped). */
int mps_drop_site(fh_ctx* ctx, fh_mps* mps, int site);

/* ---- environments (H4, H5) ---------------------------------------------
 * env_update_left : L_{site+1}[c',w',c] = sum alpha A[a',s',c']^H (L_site[a',w,a] A[a,s,c])
 * env_update_right: R_{site}[c',w,c]    = sum alpha_R conj(A[c',s',b']) R_{site+1}[b',w',b] A[c,s,b]^T
 * with alpha = recoupling coefficient (F-5) x reduced MPO element.  L_0 and R_L are the
 * boundary 1x1 blocks.  The result is stored inside the MPS object. */
int env_update_left(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, int site);
int env_update_right(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, int site);
/* which = 0: L_k, 1: R_k (k = bond index).  Layout query and download as for sites:
 * labels[nblk][5] = (qx',tjx',w,qx,tjx), dims[nblk][2]. */
int env_layout(const fh_mps* mps, int which, int bond, int* nblk, int64_t* nelem, int32_t* labels,
               int32_t* dims);
int env_get(fh_ctx* ctx, const fh_mps* mps, int which, int bond, void* data, int64_t capacity_elems, int data_is_device);
int env_set(fh_ctx* ctx, fh_mps* mps, int which, int bond, int nblk, const int32_t* labels,
            const void* data, int data_is_device);

/* ---- hot path: H_eff theta = L . W_i . W_{i+1} . theta . R  (H0-H3) --
 * heff_plan emits the two task lists of the apply on bond (site, site+1) [nsite = 2] or on
 * site `site` [nsite = 1] from the sector tables, MPO sparsity and recoupling coefficients,
 * sorts them canonically, builds the tile queue and uploads everything.  It uses L_site and
 * R_{site+nsite} stored in the MPS. */
int heff_plan(fh_ctx* ctx, const fh_mpo* mpo, const fh_mps* mps, int site, int nsite);
/* Interchange format of the vector H_eff acts on: nsite=2: labels[nblk][8] = (qa,tja,s1,qc,tjc,s2,qb,tjb);
 * nsite=1: labels[nblk][5].  dims[nblk][2].  The blocks in this (canonical) order, each dense row-major, one
 * after the other, plain tensor entries: nelem complex128 in all. */
int heff_layout(const fh_ctx* ctx, int* nblk, int64_t* nelem, int32_t* labels, int32_t* dims);
/* host copy of a task list, stage = 1 or 2: tuples[ntask][3] = (out_id, lhs_id, rhs_id), ids =
 * positions in canonical block order (stage 1: Z, L, theta; stage 2: out, Z, R); alpha[ntask].
 * Pass tuples = alpha = NULL to query ntask (and nout = number of output blocks).  An intermediate block
 * that no stage-2 task reads is not part of the lists (reading A-17). */
int heff_get_tasks(const fh_ctx* ctx, int stage, int* ntask, int* nout, int32_t* tuples, double* alpha);
/* Planned vectors.  heff_apply / heff_inner / heff_expm work on device vectors of heff_layout's nelem
 * complex128 in the library's PLANNED layout, which is opaque: for nsite = 2 the blocks that share the middle
 * label c form one row-major matrix theta_c[(a,s1,alpha),(s2,b,beta)] (the matrix the SVD split factorises,
 * PAPER.md:250; a whole row panel is then one GEMM operand) and every entry carries the factor sqrt(2 j_b + 1),
 * which turns the multiplet-weighted inner product F-6 into the plain Euclidean one; for nsite = 1 it equals
 * the interchange format.  heff_import / heff_export convert on the device (one scaled block-copy kernel,
 * H8 type); source and destination must not overlap. */
int heff_import(fh_ctx* ctx, const void* blocks_dev, void* vec_dev);
int heff_export(fh_ctx* ctx, const void* vec_dev, void* blocks_dev);
/* out_dev = H_eff * theta_dev; both planned device vectors. */
int heff_apply(fh_ctx* ctx, const void* theta_dev, void* out_dev);
/* Same operation with HOST buffers (pageable or pinned) of heff_layout's nelem complex128 in the INTERCHANGE
 * format: copies theta to the device, imports, applies, exports, copies the result back and synchronises
 * the stream.  This is the end-to-end entry a caller without device memory uses. */
int heff_apply_host(fh_ctx* ctx, const void* theta_host, void* out_host);
/* sum over both task lists of 8*m*n*k */
int64_t heff_flops(const fh_ctx* ctx);
/* <x,y> of two planned vectors = sum_blocks (2 j_b + 1) sum conj(x) y of the tensors they hold (F-6);
 * result[2] = re,im */
int heff_inner(fh_ctx* ctx, const void* x_dev, const void* y_dev, double* result);
/* out_dev = exp(-i tau H_eff) theta_dev by an m-vector Lanczos process (H6, H7) */
int heff_expm(fh_ctx* ctx, const void* theta_dev, void* out_dev, double tau, int krylov_dim);
/* Same with the adaptive stop of reading A-15: at most krylov_dim vectors, stop when the
 * residual estimate is <= adapt_tol (> 0); *k_used (host, may be NULL) receives the number of vectors used.
 * One stream synchronisation per Lanczos step. */
int heff_expm_adaptive(fh_ctx* ctx, const void* theta_dev, void* out_dev, double tau, int krylov_dim,
                       double adapt_tol, int* k_used);
/* cumulative since context creation, sector matrices factorised (H9 and the one-site splits) by route:
 * counts[0] own shared-memory Jacobi kernel (matrix and V fit 216 KB: up to 82 x 82), [1] cusolverDnXgesvdp, [2] cusolverDnZgesvd
 * (n < 48, or redo of [3]), [3] gesvdp results rejected because it reported a perturbed spectrum,
 * [4] Householder QR by cusolverDnZgeqrf + Zungqr (one-site splits that do not fit shared memory), [5] Householder
 * QR by the library's own shared-memory kernel, [6] own global-memory Jacobi kernel (matrices above the
 * shared-memory route with at most 128 columns; it runs on a side stream beside the vendor routines), [7] Gram-matrix
 * eigenvalue route (G = B^H B, cusolverDnZheevd, U = B V / sigma; FH_OPT_SVD_GRAM_MINN), [8] sectors of [7] redone by
 * the vendor SVD because the truncation kept a singular value below 3e-3 of the sector's largest. */
int fh_factorization_stats(const fh_ctx* ctx, int64_t counts[9]);
/* Task-list cache of the one-site sweeps (H0).  One-site TDVP keeps every bond's sector table
 * (no SVD, bond dimension fixed), so tdvp1_sweep / tdvp_sweep_auto keep the task lists they emit in
 * host memory owned by the fh_mps and reuse an entry only when the labels and shapes of every tensor the emitter
 * reads, and the MPO's t_h and U, are identical to those it was emitted for; a two-site sweep empties the cache.
 * Results do not depend on it (same lists, same launches).  Stats: lookups that reused / re-emitted a list since
 * the state was created, and the host bytes held now (any pointer may be NULL).  Limit: drops all entries and
 * caps the host memory of new ones (default 4 GiB; 0 switches the cache off).  Host-only calls; FH_EINVAL on a
 * NULL state or a negative limit. */
int fh_plan_cache_stats(const fh_mps* mps, int64_t* hits, int64_t* misses, int64_t* host_bytes);
int fh_plan_cache_limit(fh_mps* mps, int64_t max_host_bytes);
/* cumulative since context creation: exponentials evaluated and Krylov vectors (= H_eff applies) they used */
int fh_krylov_stats(const fh_ctx* ctx, int64_t* n_exponentials, int64_t* n_vectors);

/* ---- time evolution ---------------------------------------------------
 * One full step dt = left->right half-sweep with tau = dt/2 followed by right->left with
 * tau = dt/2 (reading A-4); at every bond: merge, Lanczos exponential, block-wise SVD with the
 * truncation rule A-6, environment update, one-site backward step. */
typedef struct {
  int krylov_dim;      /* Lanczos vectors m (>= 2) */
  double krylov_tol;   /* happy-breakdown threshold on beta_j (relative to 1), e.g. 1e-12 */
  int chi_max_full;    /* cap on sum d (2j+1) of the new bond */
  double eps_trunc;    /* discarded relative weight; < 0 disables */
  double krylov_adapt_tol; /* > 0: adaptive Krylov dimension (reading A-15): stop after k <= krylov_dim
                            * vectors once |tau| beta_k |e_k^T exp(-i tau T_k) e_1| <= krylov_adapt_tol (residual of
                            * the Krylov approximation in y' = -i H y, times the step; relative to |theta|).
                            * <= 0: always krylov_dim vectors (BASELINE config 3). */
} fh_params;
int tdvp2_sweep(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, double dt, const fh_params* params);
/* One full ONE-site TDVP time step dt ("switch from the two-site to the one-site TDVP
 * update once the bond dimension has saturated"): L->R half-sweep then R->L, tau = dt/2; at every site:
 * forward one-site Lanczos step, split without truncation (block-wise SVD of the (a,s)-stacked or
 * (s,b)-side-by-side blocks), environment update, backward ZERO-site step on the bond matrix
 * (K C = sum_w L C R^T, recoupling coefficient 1), absorption into the next site.  Bond dimensions
 * never grow.  Preconditions and state on return as tdvp2_sweep (centre on site 0, right environments
 * built); krylov_dim and krylov_tol of params are used, chi_max_full and eps_trunc are not. */
int tdvp1_sweep(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, double dt, const fh_params* params);
/* The paper's adaptive driver (reading A-16): one full time step dt that is a two-site
 * step (tdvp2_sweep) until a two-site step has left the full dimension sum_c d_c (2 j_c + 1) of EVERY bond
 * no larger than before it ("the bond dimension has saturated": capped by chi_max_full in the bulk, exact at
 * the edges), and a one-site step (tdvp1_sweep) from then on; the flag lives in the fh_mps and is never
 * cleared.  *nsite_used (host, may be NULL) receives 2 or 1. */
int tdvp_sweep_auto(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, double dt, const fh_params* params,
                    int* nsite_used);
/* statistics of the last sweep: max discarded weight, max chi_full, max chi_su2, max d */
int tdvp2_last_stats(const fh_ctx* ctx, double* max_discarded, int* chi_full, int* chi_su2, int* dmax);

/* Singular values kept on `bond` by the most recent SVD split there (H9), concatenated sector by
 * sector in the order of mps_get_bond (d_c values per sector, descending inside a sector).  n = 0
 * if the bond has not been split yet.  Pass s = NULL to query n.  Gauge-invariant data (A-13). */
int mps_get_svals(const fh_mps* mps, int bond, int* n, double* s);

/* ---- observables (H10; reading A-12) -----------------------------------
 * n_i = <1> ratio (== 1 in a T_tot = 0 state), sz_i = <S^z_i>, docc_i = <n_up n_dn>_i = <P_D>/2;
 * host arrays of length L.  Requires all sites right of the centre right-canonical (true
 * after mps_init_neel / tdvp2_sweep). */
int measure_local(fh_ctx* ctx, const fh_mps* mps, double* n_i, double* sz_i, double* docc_i);
/* <psi|psi> and <psi|H|psi>/<psi|psi> by a full left contraction */
int measure_global(fh_ctx* ctx, const fh_mpo* mpo, const fh_mps* mps, double* norm2, double* energy);

/* seconds spent (CUDA events on the context stream) since the last fh_reset_timers, by phase */
int fh_get_timers(const fh_ctx* ctx, double* sec_heff, double* sec_env, double* sec_svd,
                  double* sec_vec, double* sec_pack);
int fh_reset_timers(fh_ctx* ctx);
/* algorithmic bytes the HBM-bound phases moved since the last fh_reset_timers: vec = Lanczos vector kernels (H6:
 * 32 n per dot, 64 n per three-term update, 16 (m+1) n per linear combination), pack = pack / unpack around the
 * SVD (H8: 32 bytes per element + the zero fill).  With fh_get_timers: GB/s of those kernels inside a sweep. */
int fh_get_traffic(const fh_ctx* ctx, int64_t* vec_bytes, int64_t* pack_bytes);
/* on = 0: the library records no phase events any more (fh_get_timers then returns what was accumulated before);
 * on != 0 (the default at context creation) records them again.  An event record between two kernels of the
 * Lanczos loop costs about a microsecond of GPU time and keeps the next kernel from being set up while its
 * predecessor drains, so production runs that do not read the breakdown switch the timers off. */
int fh_enable_timers(fh_ctx* ctx, int on);
/* number of kernels the library launched since context creation */
int64_t fh_launch_count(const fh_ctx* ctx);

/* ---- calibration helper for the roofline denominator ------------------------
 * Runs cublasZgemm (is_complex=1) or cublasDgemm n x n x n `reps` times on the context stream
 * and returns the average seconds per call.  Library GEMM, not part of the hot path. */
int fh_cublas_gemm_seconds(fh_ctx* ctx, int n, int is_complex, int reps, double* seconds);

/* FP64 tensor-pipe issue peak: a register-only loop of DMMA.8x8x4 (mma.sync.m8n8k4.f64) on every
 * SM; returns the achieved TFLOP/s (2 flops per FMA).  The roofline denominator of the GEMM
 * kernels, measured on the same device and clocks as the run.  Not part of the hot path. */
int fh_dmma_peak_tflops(fh_ctx* ctx, int reps, double* tflops);

/* ---- Lanczos vector kernels and scaled block copy on caller data (H6, H8) ---------------------------------
 * The kernels expm_lanczos and the pack / unpack steps launch, callable on their own.  A vector of n complex128
 * is a sequence of nblk contiguous blocks of blk_len[b] elements with the integer weight blk_weight[b] (= 2j+1);
 * the library cuts it into chunks of the length it would use for a Krylov vector of that size (1024 / 2048 /
 * 8192 elements below 1 Mi / below 4 Mi / above).  Reductions run in a fixed order (bit-identical results).
 *   fh_vec_wdot:            result = sum_b weight_b sum conj(x) y                       (F-6; one launch)
 *   fh_vec_lanczos_update:  the three-term recurrence on UNNORMALISED Krylov vectors u_j = b_j v_j:
 *                           w <- (w - (a_raw / bj2) u_j) / sqrt(bj2) - sqrt(bj2 / bjm2) u_prev,  *norm2_out = <w,w>;
 *                           bj2 <= 0 means b_j = 1, uprev_dev NULL or bjm2 <= 0 drops the u_prev term; a norm below
 *                           tol gives a zero reciprocal (happy breakdown)
 *   fh_vec_lincomb:         y = sum_j coef_j V[j * stride + .]  (coef = m complex numbers as 2m doubles, m <= 32)
 *   fh_copy_blocks:         dst[dst_off + r ld_dst + c] (or [c ld_dst + r] if transpose) = scale * src[src_off + r ld_src + c]
 * All pointers named _dev are device pointers; the other arrays are host arrays of nblk entries. */
int fh_vec_wdot(fh_ctx* ctx, int64_t n, int nblk, const int64_t* blk_len, const int32_t* blk_weight, const void* x_dev,
                const void* y_dev, double* result);
int fh_vec_lanczos_update(fh_ctx* ctx, int64_t n, int nblk, const int64_t* blk_len, const int32_t* blk_weight, double a_raw,
                          double bj2, double bjm2, double tol, const void* uj_dev, const void* uprev_dev, void* w_dev,
                          double* norm2_out);
int fh_vec_lincomb(fh_ctx* ctx, int64_t n, int m, const double* coef, const void* V_dev, int64_t stride, void* y_dev);
/* The split-precision segmented complex GEMM of FH_OPT_PRECISION = 1 on caller data (
 * PAPER.md:264-270; oracle/splitprec.py): one output block
 *     C (M x N, row-major, leading dimension ldc) = sum_t alpha[t] op(A_t) (M x K[t]) B_t (K[t] x N),
 *     op(A_t)(m, k) = A_dev[a_off[t] + m a_sm[t] + k a_sk[t]]   (conjugated if conj_a),
 *     B_t(k, n)     = B_dev[b_off[t] + k b_sk[t] + n b_sn[t]]
 * (offsets and strides in complex128 elements; host arrays of nseg entries; nseg = 0 stores zeros), every product
 * taken as 3 x TF32 on tcgen05 with float32 accumulation in tensor memory.  A_dev, B_dev, C_dev are device
 * pointers to complex128; C must not overlap A or B.  Returns after the kernel has finished. */
int fh_zgemm_split(fh_ctx* ctx, int M, int N, int nseg, const int32_t* K, const double* alpha, int conj_a, const void* A_dev,
                   const int64_t* a_off, const int32_t* a_sm, const int32_t* a_sk, const void* B_dev, const int64_t* b_off,
                   const int32_t* b_sk, const int32_t* b_sn, void* C_dev, int ldc);
int fh_copy_blocks(fh_ctx* ctx, int nblk, const int64_t* src_off, const int64_t* dst_off, const int32_t* rows, const int32_t* cols,
                   const int32_t* ld_src, const int32_t* ld_dst, const int32_t* transpose, const double* scale,
                   const void* src_dev, void* dst_dev);
/* ---- the weighted inner product without any allocation ---------------------------------------------------------
 * fh_vec_wdot_static computes what fh_vec_wdot computes,
 *     result = sum_b blk_weight[b] * sum_{i in block b} conj(x_i) y_i          (F-6; the reduction of H6),
 * for callers that may not call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it).  It needs no context, calls no cudaMalloc / cudaFree / allocating library routine, does not
 * synchronise and copies nothing to the host: two kernel launches on the caller's stream.
 *   n, nblk            vector length in complex128 elements and number of blocks: 1 <= nblk <=
 *                      FH_STATIC_MAX_BLOCKS, 1 <= n <= FH_STATIC_MAX_ELEMS; beyond that FH_EINVAL, nothing launched
 *   blk_len_dev        DEVICE array of nblk int64 block lengths (>= 0, sum = n; a table that breaks this makes
 *                      the result NaN + i NaN), blk_weight_dev DEVICE array of nblk int32 weights (2j+1)
 *   x_dev, y_dev       DEVICE vectors of n complex128 (interleaved re, im); not written
 *   result_dev         DEVICE, 2 doubles (re, im), written by the second kernel; owned by the caller
 *   stream             the caller's cudaStream_t (NULL = the default stream)
 * Its scratch memory (block prefix offsets, one partial sum per CTA, a retirement counter) is ONE file-scope
 * device array of FH_STATIC_SCRATCH_BYTES bytes, which every GPU that loads the library holds until the process
 * exits.  All calls share it and it keeps the last call's contents (each call clears what it needs cleared):
 * calls that overlap on one GPU -- streams without an ordering between them, several host threads -- race on it;
 * the caller orders them.  The sum is taken per CTA over contiguous 1024-element ranges (longer ones beyond 4 Mi
 * elements) and then over the CTAs in index order: deterministic, and equal to fh_vec_wdot up to the rounding of a
 * different summation order.
 * fh_static_setup takes the device address of the array for the CURRENT device (cudaGetSymbolAddress, once per
 * device); fh_vec_wdot_static calls it on first use on a device -- call it yourself before a graph capture
 * starts.  fh_static_last_error: message of the last failed call of these two on the calling thread. */
#define FH_STATIC_MAX_BLOCKS 16384
#define FH_STATIC_MAX_ELEMS ((int64_t)1 << 32)
#define FH_STATIC_SCRATCH_BYTES 196872
int fh_static_setup(void);
int fh_vec_wdot_static(int64_t n, int nblk, const int64_t* blk_len_dev, const int32_t* blk_weight_dev, const void* x_dev,
                       const void* y_dev, double* result_dev, void* stream);
const char* fh_static_last_error(void);

/* HBM-bound kernels of the path timed in isolation on n_elems complex128
 * elements taken from the arena (FH_ENOMEM if (m + 3) * n_elems do not fit): gbs[0] weighted dot (one launch,
 * last CTA sums the partials), gbs[1] axpy, gbs[2] scale, gbs[3] m-vector linear combination, gbs[4] pack
 * (scaled block copy, 256 x 256 blocks), gbs[5] pack with transposition, gbs[6] the Lanczos three-term update
 * w -= alpha v_j + beta v_{j-1} fused with <w,w>.  GB/s = algorithmic bytes (32 n, 48 n, 32 n, 16 (m+1) n,
 * 32 n, 32 n, 64 n) / CUDA-event time averaged over reps; gbs has 7 entries.  Measurement helper, not on
 * the path. */
int fh_vec_kernels_gbs(fh_ctx* ctx, int64_t n_elems, int m, int reps, double* gbs);

/* F-6: w(c,b) = sqrt((2 j_b + 1) / (2 j_c + 1)), the weight under which a site tensor A[c,s,b] is right-canonical,
 * sum_{s,b} w^2 A A^H = 1 (doubled spins tjc, tjb).  Host only. */
double fh_canonical_weight(int tjc, int tjb);
/* ---- host-only entry points (no CUDA call inside): the symmetry layer on its own -----------
 * Closed-form recoupling coefficients of reading F-5 (all arguments doubled spins):
 *   coefL(a,s,c; k,r,k'; a',s',c') = sqrt((2c+1)(2k'+1)(2a'+1)(2s'+1)) {a s c; k r k'; a' s' c'}
 *   coefR(c,s,b; k,r,k'; c',s',b') = (2b'+1)/(2c'+1) sqrt((2b+1)(2k'+1)(2c'+1)(2s'+1)) {c s b; k r k'; c' s' b'} */
double fh_coef_left(int ta, int ts, int tc, int tk, int tr, int tkp, int tap, int tsp, int tcp);
double fh_coef_right(int tc, int ts, int tb, int tk, int tr, int tkp, int tcp, int tsp, int tbp);
/* label algebra fh_host_plan uses (host-only twin of FH_OPT_SYMMETRY): 0 = U(1) x SU(2), 1 = U(1) x U(1) */
int fh_host_set_symmetry(int mode);
/* Emit the task lists of an apply on `site` (nsite = 1 | 2; nsite = 0: the zero-site apply of one-site
 * TDVP on the bond whose bra-side dims are bl and ket-side dims br) from explicit tables: bl/br =
 * [n][3] (q,tj,d) of the left and right bond, Llab/Rlab = [nblk][5] canonical-order labels of the
 * environment blocks.  Results are kept in a process-global scratch (not thread-safe) and read
 * with fh_host_get_tasks (same format as heff_get_tasks; flops = sum 8mnk of that stage). */
int fh_host_plan(int site, int nsite, double t_h, double U, int nl, const int32_t* bl, int nr, const int32_t* br,
                 int nLblk, const int32_t* Llab, int nRblk, const int32_t* Rlab);
int fh_host_get_tasks(int stage, int* ntask, int* nout, int32_t* tuples, double* alpha, int64_t* flops);
/* Warp-unit list of the same host plan (what the grouped ZGEMM launches): per unit
 * [out, m0, n0, mt, nt, steps] (int32[nunit][6], launch order = heaviest first) and per output block
 * [M, N, steps] (int32[nout][3]); dmma_padded = DMMA.8x8x4 instructions the list issues.  Either array
 * pointer may be NULL to query the counts only. */
int fh_host_get_units(int stage, int* nunit, int32_t* units, int* nout, int32_t* outs, int64_t* dmma_padded);
/* Tile list of the split-precision kernel (zgemm_tc.cu, NEXT-3) for the same host plan and `grid` persistent CTAs:
 * per tile [out, m0, n0, h, w, chunks] (int32[ntile][6]; out indexes the merged outputs of fh_host_get_units, a tile
 * is h x w <= 128 x 128 elements of it, chunks = sum over its segments of ceil(K / 16)), in the order the kernel walks
 * them: CTA b takes tiles cta_begin[b] .. cta_begin[b + 1] - 1 (int32[grid + 1]).  static_side 1 (op(A)) or 2 (op(B)):
 * also the panel images of that operand: seg_img[s] = byte offset of the image segment s reads and seg_operand[s] =
 * element offset of the operand block it is made from (int64 per segment; nseg = number of segments of the stage: the
 * tasks; -1 for a segment of an output that was merged into its neighbour and is not read), nimage_chunks 32-KB chunks in image_bytes bytes; 0: skipped.  Pointers may be NULL. */
int fh_host_get_tc_tiles(int stage, int grid, int static_side, int* ntile, int32_t* tiles, int32_t* cta_begin, int* nseg,
                         int* nimage_chunks, int64_t* seg_img, int64_t* seg_operand, int64_t* image_bytes);

#ifdef __cplusplus
}
#endif
#endif /* FH_B200_H */
