// Context, arena, device pools, plans (host side of libfh_b200).
#pragma once
#include <cublas_v2.h>
#include <cusolverDn.h>

#include <future>
#include <stdexcept>

#include "fh_b200.h"
#include "symmetry.hpp"

namespace fh {

struct FhError : std::runtime_error {
  int code;
  FhError(int c, const std::string& m) : std::runtime_error(m), code(c) {}
};
#define FH_CUDA(x)                                                                                    \
  do {                                                                                                \
    cudaError_t e__ = (x);                                                                            \
    if (e__ != cudaSuccess)                                                                           \
      throw fh::FhError(FH_ECUDA, std::string(#x) + ": " + cudaGetErrorString(e__));                  \
  } while (0)
#define FH_REQUIRE(cond, code, msg) \
  do {                              \
    if (!(cond)) throw fh::FhError(code, msg); \
  } while (0)

// first-fit free-list allocator over the single HBM arena; unit = complex128 elements
struct Arena {
  int64_t cap = 0, used = 0, peak = 0;
  std::map<int64_t, int64_t> free_;  // offset -> length
  static int64_t round_up(int64_t n) { return (n + 15) / 16 * 16; }  // 256-byte granules
  void init(int64_t n) {
    cap = n;
    used = peak = 0;
    free_.clear();
    free_[0] = n;
  }
  int64_t alloc(int64_t n);
  void release(int64_t off, int64_t n);
};

// grow-only device buffer for task lists and other small per-plan tables
struct DevPool {
  char* ptr = nullptr;
  size_t cap = 0, top = 0;
  void reset() { top = 0; }
  void reserve(size_t bytes, cudaStream_t s);
  void* take(size_t bytes);
  void destroy();
};

struct Plan {
  bool valid = false;
  int nsite = 0, site = 0;
  BlockTensor vec;  // layout of the vector H_eff acts on (base unused)
  BlockTensor Z;    // stage-1 intermediate, allocated in the arena
  Stage st1, st2;
  const cplx* Lptr = nullptr;
  const cplx* Rptr = nullptr;
  std::vector<VecChunk> chunks;
  VecChunk* d_chunks = nullptr;
  double* d_partial = nullptr;
  double* d_result = nullptr;
  double* d_scal = nullptr;  // Lanczos scalars kept on the device (expm_lanczos)
  unsigned* d_counter = nullptr;  // retirement counter of the one-launch reductions (zero between launches)
  DevPool pool;
  // k-split tiles of the warp-specialised GEMM: scratch slots in the arena, arrival counters, launch number
  int64_t ws_scratch = -1, ws_scratch_n = 0;  // arena offset / elements
  unsigned* d_ws_flags = nullptr;   // one counter per scratch slot (both stages)
  unsigned* d_ws_dep = nullptr;     // one counter per stage-1 output panel (cross-stage dependencies)
  unsigned ws_epoch = 0;
  WsPair pair;                      // joint tile queue of the two stages: one launch per apply
  UnitPair upair;                   // the same for the warp-unit form (two-site plans)
  unsigned* d_unit_dep = nullptr;   // one counter per stage-1 merged output
  unsigned unit_epoch = 0;
  // interchange format <-> planned layout (heff_import / heff_export), built on first use per plan
  bool io_ready = false;
  int n_io = 0;
  CopyBlk* d_import = nullptr;
  CopyBlk* d_export = nullptr;
  DevPool io_pool;
  // tile lists of the split-precision form (FH_OPT_PRECISION = 1), built on first use per plan
  bool tc_ready = false;
  int n_tc1 = 0, n_tc2 = 0;
  fh::TcTile* d_tc1 = nullptr;
  fh::TcTile* d_tc2 = nullptr;
  int* d_tc_cb1 = nullptr;                // first tile of every persistent CTA (tiles are dealt on the host)
  int* d_tc_cb2 = nullptr;
  int64_t* d_tc_img1 = nullptr;           // per segment: byte offset of its static operand's panel images
  int64_t* d_tc_img2 = nullptr;
  unsigned char* tc_images1 = nullptr;    // stage 1: left environment as op(A); stage 2: right environment as op(B)
  unsigned char* tc_images2 = nullptr;
  DevPool tc_pool;
};

// What the emitter produces for one two-site plan; filled by a second host thread while the main thread runs
// the backward one-site step of the bond before (tdvp.cu, sweep): the emission of the next plan needs only the
// bond tables and environment layouts, which are final once the environment update has been emitted.
struct PlanEmit {
  int site = -1;
  BlockTensor vec, Z;
  Stage st1, st2;
  std::vector<VecChunk> chunks;
};

enum { T_HEFF = 0, T_ENV = 1, T_SVD = 2, T_VEC = 3, T_PACK = 4, T_NCAT = 5 };

// Task-list cache of the one-site sweeps (H0).  One-site TDVP leaves the sector tables of every bond as they
// are (no SVD, no change of bond dimension), so the task lists of a sweep equal those of the sweep
// before.  An entry holds what an emitter produced for (kind, site) together with a signature: the flattened
// labels and block shapes of every input the emitter reads, and the MPO parameters.  A lookup compares the whole
// signature, so a stale entry (a QR that lowered a rank, a two-site step in between) is re-emitted, never used.
// Task lists address operands relative to their tensor base; arena offsets may change freely between sweeps.
enum { PC_HEFF1 = 0, PC_ENVL = 1, PC_ENVR = 2, PC_HEFF0 = 3, PC_ABSORB_L = 4, PC_ABSORB_R = 5, PC_NKIND = 6 };
struct PlanCacheEntry {
  std::vector<int> sig;
  BlockTensor t0, t1;  // layouts the emitter produced (vec and Z; X and out; new A), base = -1
  Stage st1, st2;
  std::vector<VecChunk> chunks;
  size_t bytes = 0;
};
struct PlanCache {
  bool enabled = false;  // set by the one-site sweep for its own duration
  size_t bytes = 0, max_bytes = (size_t)4 << 30;  // host bytes held / cap (no new entries beyond it)
  int64_t hits = 0, misses = 0;
  std::unordered_map<int, PlanCacheEntry> map;  // kind * 65536 + site
  const PlanCacheEntry* find(int kind, int site, const std::vector<int>& sig);
  PlanCacheEntry* store(int kind, int site, std::vector<int>&& sig);  // nullptr when over the cap
  void account(PlanCacheEntry* e);  // call once the entry is filled
  void clear();
};
void sig_add(std::vector<int>& sig, const BlockTensor& t);
void sig_add(std::vector<int>& sig, const Bond& b);
void sig_add(std::vector<int>& sig, double x);

}  // namespace fh

struct fh_mpo {
  const fh::SymMode* sym = &fh::SYM_SU2;
  int L;
  double t_h, U;
  fh::MpoSite site[2];  // even / odd site parity
};

struct fh_mps {
  const fh::SymMode* sym = &fh::SYM_SU2;  // label algebra the state was created under (FH_OPT_SYMMETRY at mps_create)
  int L;
  std::vector<fh::Bond> bond;                       // L+1
  std::vector<fh::BlockTensor> A, Lenv, Renv;       // L, L+1, L+1
  std::vector<std::vector<double>> sval;            // L+1: kept singular values of the last split
  bool saturated = false;                           // tdvp_sweep_auto: a two-site step grew no bond (A-16)
  mutable fh::PlanCache cache;                      // task lists of the one-site sweeps (host memory only)
};

struct fh_ctx {
  cudaStream_t stream = nullptr;
  fh::cplx* arena = nullptr;
  bool own_arena = false;
  fh::Arena alloc;
  std::string err;
  fh::Plan plan;
  fh::PlanEmit prefetch;           // next two-site plan, emitted ahead (see PlanEmit)
  std::future<void> prefetch_job;
  bool prefetch_pending = false;
  int64_t prefetch_used = 0;
  fh::DevPool pool_aux;  // env updates, merge, pack, measure
  fh::DevPool pool_small;  // descriptors of the small-matrix SVD kernel
  int64_t launches = 0;
  // algorithmic bytes of the HBM-bound phases since the last fh_reset_timers (H6: 32 n per dot, 64 n per three-term
  // update, 16 (m + 1) n per linear combination; H8: 32 bytes per packed / unpacked element): with the phase
  // timers they give the GB/s those kernels reach INSIDE a sweep
  int64_t vec_bytes = 0, pack_bytes = 0;
  // pinned host scratch
  double* h_pinned = nullptr;  // 4096 doubles
  size_t h_pinned_n = 0;
  // timers (event pairs around every phase; fh_enable_timers(ctx, 0) drops them: an event record between two
  // kernels costs GPU front-end time and cancels the programmatic dependent launch across it)
  bool timers_on = true;
  bool span_open = false;
  double sec[fh::T_NCAT] = {0, 0, 0, 0, 0};
  struct Span {
    cudaEvent_t a, b;
    int cat;
  };
  std::vector<Span> spans;
  std::vector<cudaEvent_t> ev_free;
  // SVD (H9): one cuSOLVER handle + stream + workspace per host worker thread; the sector SVDs of a
  // bond are independent and cuSOLVER's SVD drivers block their calling thread, so concurrency needs
  // host threads (tdvp.cu, run_sector_svds)
  struct SvdWorker {
    cusolverDnHandle_t h = nullptr;
    cusolverDnParams_t params = nullptr;
    cublasHandle_t cb = nullptr;          // Gram / back-multiplication GEMMs of the eigenvalue route (tdvp.cu, svd_one)
    cudaStream_t s = nullptr;
    void* dwork = nullptr;
    size_t dwork_bytes = 0;
    std::vector<char> hwork;
    int* d_info = nullptr;
    cudaEvent_t done = nullptr;
  };
  std::vector<SvdWorker> svd_workers;
  cudaEvent_t svd_fork = nullptr;
  cudaStream_t svd_side = nullptr;       // mid_svd_kernel runs here, beside the main stream and the workers
  cudaEvent_t svd_side_done = nullptr;
  int64_t svd_mid = 0;                   // sector matrices factorised by mid_svd_kernel
  cudaEvent_t small_copied = nullptr;  // descriptors of the small-matrix kernels have left small_desc_host
  bool small_copied_armed = false;
  std::vector<char> small_desc_host;
  int device = 0;
  const fh::SymMode* sym = &fh::SYM_SU2;  // fh_set_option(FH_OPT_SYMMETRY): the label algebra of every object of the context
  int opt_gemm_path = 0;      // fh_set_option: 0 auto, 1 warp units (two launches), 2 warp-specialised, 3 warp units (one launch)
  int opt_svd_mid_maxn = 100;
  int opt_svd_small_maxn = 4096;
  int opt_svd_threads = 0;    // 0 = default
  int opt_svd_gram_minn = 104;  // fh_set_option(FH_OPT_SVD_GRAM_MINN): narrowest sector matrix (columns) of the vendor route that
                                // goes through the Gram-matrix eigenvalue route (0 = never)
  int opt_svd_gram_batch_maxn = 256;  // fh_set_option(FH_OPT_SVD_GRAM_BATCH_MAXN): widest Gram-route sector that joins the batched eigensolver call
  int opt_precision = 0;      // fh_set_option(FH_OPT_PRECISION): 0 = FP64 DMMA, 1 = 3 x TF32 on tcgen05 (two-site applies)
  int num_sms = 148;
  unsigned* d_ws_counters = nullptr;  // tile-queue head and retired-CTA count of the warp-specialised GEMM (zero between launches)
  // status words of the last batch of sector factorisations (one per matrix, + one more per matrix for the
  // second vendor call of a QR): 0 = fine, otherwise a cuSOLVER devInfo or FACT_NOT_CONVERGED from a Jacobi kernel
  int* d_fact_status = nullptr;
  int* h_fact_status = nullptr;  // pinned
  int fact_status_cap = 0, fact_status_n = 0;
  bool fact_status_pending = false;
  int64_t svd_count[4] = {0, 0, 0, 0};  // gesvd, gesvdp, gesvdp fallbacks to gesvd, Gram-matrix eigenvalue route
  int64_t svd_gram_redone = 0;           // Gram-route sectors redone by the vendor SVD (a kept singular value too small)
  int64_t qr_small = 0;  // one-site splits done by small_qr_kernel
  int64_t svd_small = 0, qr_count = 0;  // sector matrices done by small_svd_kernel / by geqrf+ungqr
  int64_t krylov_calls = 0, krylov_vectors = 0;  // exponentials evaluated / Krylov vectors (= H_eff applies) used
  // last sweep statistics
  double stat_disc = 0.0;
  int stat_chi = 0, stat_su2 = 0, stat_dmax = 0;

  fh::cplx* ptr(int64_t off) const { return arena + off; }
  void alloc_tensor(fh::BlockTensor& t);
  void free_tensor(fh::BlockTensor& t);
  void timer_begin(int cat);
  void timer_end();
  void timers_resolve();
  void ensure_pinned(size_t ndoubles);
};

namespace fh {
// arena scratch that is returned when the scope is left, also by an exception
struct ArenaScratch {
  fh_ctx* ctx;
  int64_t off, n;
  ArenaScratch(fh_ctx* c, int64_t nelem) : ctx(c), off(c->alloc.alloc(nelem)), n(nelem) {}
  ~ArenaScratch() { ctx->alloc.release(off, n); }
  ArenaScratch(const ArenaScratch&) = delete;
  ArenaScratch& operator=(const ArenaScratch&) = delete;
  cplx* ptr() const { return ctx->ptr(off); }
};
template <class T>
T* upload(DevPool& pool, const std::vector<T>& v, cudaStream_t s) {
  if (v.empty()) return nullptr;
  T* d = (T*)pool.take(v.size() * sizeof(T));
  FH_CUDA(cudaMemcpyAsync(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, s));
  return d;
}
size_t stage_bytes(const Stage& st);
void upload_stage(DevPool& pool, Stage& st, cudaStream_t s);
size_t pair_bytes(const WsPair& pr);
void upload_pair(DevPool& pool, WsPair& pr, cudaStream_t s);

// engine pieces (api.cu / tdvp.cu)
void plan_heff(fh_ctx* ctx, const fh_mpo* mpo, const fh_mps* mps, int site, int nsite);
// starts the emission of the two-site plan at `site` on another host thread (no CUDA calls there); the next
// plan_heff(site, 2) takes it over.  The caller must not change the bond tables or environment layouts the
// plan reads before that; prefetch_cancel waits for a job still in flight and drops its result.
void prefetch_plan2(fh_ctx* ctx, const fh_mpo* mpo, const fh_mps* mps, int site);
void prefetch_cancel(fh_ctx* ctx);
void apply_heff(fh_ctx* ctx, const cplx* theta, cplx* out);
void vec_import(fh_ctx* ctx, const cplx* blocks, cplx* vec);  // interchange format -> planned layout
void vec_export(fh_ctx* ctx, const cplx* vec, cplx* blocks);  // planned layout -> interchange format
double2 inner(fh_ctx* ctx, const cplx* x, const cplx* y);  // synchronises
// returns the number of Krylov vectors used; adapt_tol > 0 enables the adaptive stop (reading A-15)
int expm_lanczos(fh_ctx* ctx, cplx* theta_inout, double tau, int m, double tol, cplx* work /* (m+1)*n */,
                 double adapt_tol = 0.0);
void do_env_update_left(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, int site);
void do_env_update_right(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, int site);
void sweep(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, double dt, const fh_params* p);
void sweep1(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, double dt, const fh_params* p);
void measure_local_impl(fh_ctx* ctx, const fh_mps* mps, double* n_i, double* sz_i, double* docc_i);
// throws FH_ECUDA if a factorisation of the last batch failed; call after the stream has been synchronised
void check_fact_status(fh_ctx* ctx);
}  // namespace fh
