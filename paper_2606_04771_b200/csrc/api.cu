// C ABI entry points (include/fh_b200.h) and the engine pieces they share: arena, plans,
// H_eff apply, weighted inner product, Lanczos exponential, environment updates.
#include <cublas_v2.h>

#include <algorithm>
#include <cmath>
#include <cstring>

#include <cstdio>

#include "context.hpp"

using namespace fh;

// ============================================================================ arena / pools
int64_t Arena::alloc(int64_t n) {
  n = round_up(n < 1 ? 1 : n);
  for (auto it = free_.begin(); it != free_.end(); ++it) {
    if (it->second >= n) {
      const int64_t off = it->first, len = it->second;
      free_.erase(it);
      if (len > n) free_[off + n] = len - n;
      used += n;
      peak = std::max(peak, used);
      return off;
    }
  }
  throw FhError(FH_ENOMEM, "arena exhausted: need " + std::to_string(n * 16) + " bytes, used " +
                               std::to_string(used * 16) + " of " + std::to_string(cap * 16));
}
void Arena::release(int64_t off, int64_t n) {
  n = round_up(n < 1 ? 1 : n);
  used -= n;
  auto it = free_.emplace(off, n).first;
  auto nx = std::next(it);
  if (nx != free_.end() && it->first + it->second == nx->first) {
    it->second += nx->second;
    free_.erase(nx);
  }
  if (it != free_.begin()) {
    auto pv = std::prev(it);
    if (pv->first + pv->second == it->first) {
      pv->second += it->second;
      free_.erase(it);
    }
  }
}

void DevPool::reserve(size_t bytes, cudaStream_t s) {
  top = 0;
  if (bytes <= cap) return;
  if (ptr) {
    FH_CUDA(cudaStreamSynchronize(s));
    FH_CUDA(cudaFree(ptr));
  }
  cap = bytes + bytes / 2 + 4096;
  FH_CUDA(cudaMalloc((void**)&ptr, cap));
}
void* DevPool::take(size_t bytes) {
  const size_t b = (bytes + 255) / 256 * 256;
  if (top + b > cap) throw FhError(FH_ENOMEM, "device pool overflow");
  void* p = ptr + top;
  top += b;
  return p;
}
void DevPool::destroy() {
  if (ptr) cudaFree(ptr);
  ptr = nullptr;
  cap = top = 0;
}

size_t fh::stage_bytes(const Stage& st) {
  return st.segs.size() * sizeof(GemmSeg) + st.units.size() * sizeof(GemmUnit) + st.tiles.size() * sizeof(WsTile) + 6 * 256;
}
size_t fh::pair_bytes(const WsPair& pr) {
  return pr.tiles.size() * sizeof(WsTile) + pr.segs.size() * sizeof(GemmSeg) + pr.dep_id.size() * 8 +
         (size_t)(pr.n_slots + pr.n_dep_counters) * sizeof(unsigned) + 8 * 256;
}
void fh::upload_pair(DevPool& pool, WsPair& pr, cudaStream_t s) {
  pr.d_tiles = upload(pool, pr.tiles, s);
  pr.d_segs = upload(pool, pr.segs, s);
  pr.d_dep_id = upload(pool, pr.dep_id, s);
  pr.d_dep_target = upload(pool, pr.dep_target, s);
}
void fh::upload_stage(DevPool& pool, Stage& st, cudaStream_t s) {
  st.d_segs = upload(pool, st.segs, s);
  st.d_units = upload(pool, st.units, s);
  st.d_tiles = upload(pool, st.tiles, s);
}

void fh_ctx::alloc_tensor(BlockTensor& t) { t.base = alloc.alloc(t.nelem); }
void fh_ctx::free_tensor(BlockTensor& t) {
  if (t.base >= 0) alloc.release(t.base, t.nelem);
  t.base = -1;
}
void fh_ctx::ensure_pinned(size_t n) {
  if (n <= h_pinned_n) return;
  if (h_pinned) {
    FH_CUDA(cudaStreamSynchronize(stream));
    FH_CUDA(cudaFreeHost(h_pinned));
  }
  h_pinned_n = n * 2 + 1024;
  FH_CUDA(cudaMallocHost((void**)&h_pinned, h_pinned_n * sizeof(double)));
}
void fh_ctx::timer_begin(int cat) {
  if (span_open) timer_end();  // a span left open by an exception: close it here so that both events exist
  span_open = timers_on;
  if (!timers_on) return;
  if (spans.size() > 8192) timers_resolve();
  Span sp;
  for (cudaEvent_t* e : {&sp.a, &sp.b}) {
    if (!ev_free.empty()) {
      *e = ev_free.back();
      ev_free.pop_back();
    } else {
      FH_CUDA(cudaEventCreate(e));
    }
  }
  sp.cat = cat;
  FH_CUDA(cudaEventRecord(sp.a, stream));
  spans.push_back(sp);
}
void fh_ctx::timer_end() {
  if (!span_open) return;
  span_open = false;
  FH_CUDA(cudaEventRecord(spans.back().b, stream));
}
void fh_ctx::timers_resolve() {
  if (spans.empty()) return;
  FH_CUDA(cudaStreamSynchronize(stream));
  if (span_open) timer_end();
  FH_CUDA(cudaStreamSynchronize(stream));
  for (Span& sp : spans) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, sp.a, sp.b) == cudaSuccess) sec[sp.cat] += ms * 1e-3;
    else cudaGetLastError();  // a span whose end was never recorded (error path): dropped, not fatal
    ev_free.push_back(sp.a);
    ev_free.push_back(sp.b);
  }
  spans.clear();
}

// ============================================================================ task-list cache (one-site sweeps)
void fh::sig_add(std::vector<int>& sig, const BlockTensor& t) {
  const size_t n = t.keys.size();
  sig.push_back(t.nlab);
  sig.push_back((int)n);
  const size_t at = sig.size();
  sig.resize(at + n * 14);
  int* p = sig.data() + at;
  for (size_t i = 0; i < n; ++i) {
    std::memcpy(p, t.keys[i].data(), 12 * sizeof(int));
    p[12] = t.rows[i];
    p[13] = t.cols[i];
    p += 14;
  }
}
void fh::sig_add(std::vector<int>& sig, const Bond& b) {
  sig.push_back((int)b.sec.size());
  for (size_t i = 0; i < b.sec.size(); ++i) {
    sig.push_back(b.sec[i].q);
    sig.push_back(b.sec[i].tj);
    sig.push_back(b.d[i]);
  }
}
void fh::sig_add(std::vector<int>& sig, double x) {
  int w[2];
  std::memcpy(w, &x, sizeof(double));
  sig.push_back(w[0]);
  sig.push_back(w[1]);
}
const PlanCacheEntry* PlanCache::find(int kind, int site, const std::vector<int>& sig) {
  auto it = map.find(kind * 65536 + site);
  if (it != map.end() && it->second.sig == sig) {
    ++hits;
    return &it->second;
  }
  ++misses;
  return nullptr;
}
PlanCacheEntry* PlanCache::store(int kind, int site, std::vector<int>&& sig) {
  auto it = map.find(kind * 65536 + site);
  if (it != map.end()) {
    bytes -= std::min(bytes, it->second.bytes);
    map.erase(it);
  }
  if (bytes >= max_bytes) return nullptr;
  PlanCacheEntry& e = map[kind * 65536 + site];
  e.sig = std::move(sig);
  return &e;
}
static size_t stage_host_bytes(const Stage& st) {
  return st.t_out.size() * (3 * sizeof(int) + sizeof(double)) + st.outs.size() * sizeof(GemmOut) +
         st.segs.size() * sizeof(GemmSeg) + st.units.size() * sizeof(GemmUnit);
}
static size_t layout_host_bytes(const BlockTensor& t) { return t.keys.size() * (sizeof(Key) * 2 + 48); }
void PlanCache::account(PlanCacheEntry* e) {
  e->bytes = e->sig.size() * sizeof(int) + stage_host_bytes(e->st1) + stage_host_bytes(e->st2) +
             layout_host_bytes(e->t0) + layout_host_bytes(e->t1) + e->chunks.size() * sizeof(VecChunk);
  bytes += e->bytes;
}
void PlanCache::clear() {
  map.clear();
  bytes = 0;
}

// ============================================================================ plan + apply
static int last_tj_pos(int nsite) { return nsite == 2 ? 7 : (nsite == 1 ? 4 : 1); }

// weighted inner-product chunks (F-6)
static void fill_chunks(const BlockTensor& vec, int tpos, std::vector<VecChunk>& chunks) {
  chunks.clear();
  const int cl = vec_chunk_len(vec.nelem);
  if (tpos < 0) {  // two-site vector: held as sqrt(2 j_b + 1) theta, so F-6 is the plain Euclidean product
    for (int64_t s = 0; s < vec.nelem; s += cl)
      chunks.push_back(VecChunk{s, (int)std::min<int64_t>(cl, vec.nelem - s), 1.0f});
    return;
  }
  for (size_t i = 0; i < vec.keys.size(); ++i) {
    const int64_t n = (int64_t)vec.rows[i] * vec.cols[i];
    for (int64_t s = 0; s < n; s += cl)
      chunks.push_back(VecChunk{vec.off[i] + s, (int)std::min<int64_t>(cl, n - s), (float)(vec.keys[i][tpos] + 1)});
  }
}
// host-only emission of the two-site plan at `site` (no CUDA calls: also runs on the prefetch thread)
static void emit_plan2(const fh_mpo* mpo, const fh_mps* mps, int site, BlockTensor& vec, BlockTensor& Z, Stage& st1,
                       Stage& st2, std::vector<VecChunk>& chunks) {
  layout_theta(mps->bond[site], mps->bond[site + 2], vec);
  emit_heff2(mps->Lenv[site], mps->Renv[site + 2], vec, mpo->site[site & 1], mpo->site[(site + 1) & 1], Z, st1, st2);
  fill_chunks(vec, -1, chunks);
}
void fh::prefetch_plan2(fh_ctx* ctx, const fh_mpo* mpo, const fh_mps* mps, int site) {
  prefetch_cancel(ctx);
  if (site < 0 || site + 2 > mps->L || mps->Lenv[site].base < 0 || mps->Renv[site + 2].base < 0) return;
  PlanEmit* e = &ctx->prefetch;
  e->site = site;
  const SymMode* mode = ctx->sym;
  ctx->prefetch_job = std::async(std::launch::async, [mpo, mps, site, e, mode]() {
    SymScope scope(mode);
    e->Z.base = -1;
    emit_plan2(mpo, mps, site, e->vec, e->Z, e->st1, e->st2, e->chunks);
  });
  ctx->prefetch_pending = true;
}
void fh::prefetch_cancel(fh_ctx* ctx) {
  if (!ctx->prefetch_pending) return;
  ctx->prefetch_pending = false;
  try {
    ctx->prefetch_job.get();
  } catch (...) {
  }
}

// padded DMMAs per apply between which the warp-specialised single launch is the faster form
static const int64_t WS_MIN_DMMA = 10000000, WS_MAX_DMMA = 400000000;

void fh::plan_heff(fh_ctx* ctx, const fh_mpo* mpo, const fh_mps* mps, int site, int nsite) {
  FH_REQUIRE(nsite == 1 || nsite == 2, FH_EINVAL, "heff_plan: nsite must be 1 or 2");
  FH_REQUIRE(site >= 0 && site + nsite <= mps->L, FH_EINVAL, "heff_plan: site out of range");
  FH_REQUIRE(mpo->sym == ctx->sym && mps->sym == ctx->sym, FH_ESTATE,
             "heff_plan: MPO / MPS were created under another FH_OPT_SYMMETRY than the context has now");
  const BlockTensor& Le = mps->Lenv[site];
  const BlockTensor& Re = mps->Renv[site + nsite];
  FH_REQUIRE(Le.base >= 0 && Re.base >= 0, FH_ESTATE, "heff_plan: environments of this bond are not built");
  Plan& P = ctx->plan;
  ctx->free_tensor(P.Z);
  if (P.ws_scratch >= 0) ctx->alloc.release(P.ws_scratch, P.ws_scratch_n);
  P.ws_scratch = -1;
  P.valid = false;
  P.io_ready = false;
  P.tc_ready = false;
  P.nsite = nsite;
  P.site = site;
  const bool use_cache = nsite == 1 && mps->cache.enabled;
  std::vector<int> sig;
  const PlanCacheEntry* hit = nullptr;
  if (use_cache) {
    sig_add(sig, Le);
    sig_add(sig, Re);
    sig_add(sig, mps->bond[site]);
    sig_add(sig, mps->bond[site + 1]);
    sig_add(sig, mpo->t_h);
    sig_add(sig, mpo->U);
    hit = mps->cache.find(PC_HEFF1, site, sig);
  }
  bool prefetched = false;
  if (nsite == 2 && ctx->prefetch_pending) {
    ctx->prefetch_pending = false;
    ctx->prefetch_job.get();  // rethrows what the emitter threw
    if (ctx->prefetch.site == site) {
      P.vec = std::move(ctx->prefetch.vec);
      P.Z = std::move(ctx->prefetch.Z);
      P.st1 = std::move(ctx->prefetch.st1);
      P.st2 = std::move(ctx->prefetch.st2);
      P.chunks = std::move(ctx->prefetch.chunks);
      prefetched = true;
      ++ctx->prefetch_used;
    }
  }
  if (prefetched) {
  } else if (hit) {
    P.vec = hit->t0;
    P.Z = hit->t1;
    P.st1 = hit->st1;
    P.st2 = hit->st2;
    P.chunks = hit->chunks;
  } else {
    if (nsite == 2) {
      emit_plan2(mpo, mps, site, P.vec, P.Z, P.st1, P.st2, P.chunks);
    } else {
      layout_site(mps->bond[site], mps->bond[site + 1], P.vec);
      emit_heff1(Le, Re, P.vec, mpo->site[site & 1], P.Z, P.st1, P.st2);
      fill_chunks(P.vec, last_tj_pos(nsite), P.chunks);
    }
    if (use_cache) {
      if (PlanCacheEntry* e = mps->cache.store(PC_HEFF1, site, std::move(sig))) {
        e->t0 = P.vec;
        e->t1 = P.Z;
        e->st1 = P.st1;
        e->st2 = P.st2;
        e->chunks = P.chunks;
        mps->cache.account(e);
      }
    }
  }
  ctx->alloc_tensor(P.Z);
  // Tile queue of the warp-specialised form: only for the plans that will use it (FH_OPT_GEMM_PATH as it is NOW: set
  // it before heff_plan).  Every other plan of a sweep (one-site, and two-site plans outside the window) skips
  // the emission, the dependency lists and their upload.
  P.pair = WsPair();
  {
    const int64_t dmma = P.st1.dmma_padded + P.st2.dmma_padded;
    const bool want_ws = nsite == 2 && (ctx->opt_gemm_path == 2 || (ctx->opt_gemm_path == 0 && dmma >= WS_MIN_DMMA && dmma < WS_MAX_DMMA));
    if (want_ws) {
      emit_ws_tiles(P.st1);
      emit_ws_tiles(P.st2);
      link_stages(P.st1, P.st2, 0, P.pair);  // stage 2 reads the intermediate as its left operand
    }
  }
  P.ws_scratch_n = (int64_t)(P.st1.n_slots + P.st2.n_slots) * WS_SLOT_ELEMS;
  if (P.ws_scratch_n > 0) P.ws_scratch = ctx->alloc.alloc(P.ws_scratch_n);
  P.Lptr = ctx->ptr(Le.base);
  P.Rptr = ctx->ptr(Re.base);
  P.upair = UnitPair();
  if (nsite == 2 && ctx->opt_gemm_path == 3) link_units(P.st1, P.st2, 0, P.upair);  // only on request: measured equal or slower
  const size_t upair_bytes = P.upair.units.size() * (sizeof(GemmUnit) + sizeof(UnitLink)) + P.upair.segs.size() * sizeof(GemmSeg) +
                             P.upair.dep_id.size() * 8 + (size_t)(P.upair.n_dep_counters + 1) * sizeof(unsigned) + 8 * 256;
  const size_t need = stage_bytes(P.st1) + stage_bytes(P.st2) + pair_bytes(P.pair) + upair_bytes +
                      P.chunks.size() * (sizeof(VecChunk) + 16) + 8192;
  P.pool.reserve(need, ctx->stream);
  upload_stage(P.pool, P.st1, ctx->stream);
  upload_stage(P.pool, P.st2, ctx->stream);
  P.d_chunks = upload(P.pool, P.chunks, ctx->stream);
  P.d_partial = (double*)P.pool.take(std::max<size_t>(1, P.chunks.size()) * 2 * sizeof(double));
  P.d_result = (double*)P.pool.take(2 * sizeof(double));
  P.d_scal = (double*)P.pool.take(256 * sizeof(double));
  P.d_counter = (unsigned*)P.pool.take(sizeof(unsigned));
  FH_CUDA(cudaMemsetAsync(P.d_counter, 0, sizeof(unsigned), ctx->stream));
  upload_pair(P.pool, P.pair, ctx->stream);
  if (!P.upair.units.empty()) {
    P.upair.d_units = upload(P.pool, P.upair.units, ctx->stream);
    P.upair.d_segs = upload(P.pool, P.upair.segs, ctx->stream);
    P.upair.d_link = upload(P.pool, P.upair.link, ctx->stream);
    P.upair.d_dep_id = upload(P.pool, P.upair.dep_id, ctx->stream);
    P.upair.d_dep_target = upload(P.pool, P.upair.dep_target, ctx->stream);
    const size_t nd = (size_t)P.upair.n_dep_counters + 1;
    P.d_unit_dep = (unsigned*)P.pool.take(nd * sizeof(unsigned));
    FH_CUDA(cudaMemsetAsync(P.d_unit_dep, 0, nd * sizeof(unsigned), ctx->stream));
    P.unit_epoch = 0;
  }
  {
    const size_t nf = (size_t)P.pair.n_slots + 1, nd = (size_t)P.pair.n_dep_counters + 1;
    P.d_ws_flags = (unsigned*)P.pool.take(nf * sizeof(unsigned));
    P.d_ws_dep = (unsigned*)P.pool.take(nd * sizeof(unsigned));
    FH_CUDA(cudaMemsetAsync(P.d_ws_flags, 0, nf * sizeof(unsigned), ctx->stream));
    FH_CUDA(cudaMemsetAsync(P.d_ws_dep, 0, nd * sizeof(unsigned), ctx->stream));
  }
  P.ws_epoch = 0;
  P.valid = true;
}

// Interchange format <-> planned layout (H8-type scaled block copies).  The interchange format is what
// heff_layout describes: the blocks in canonical key order, each dense row-major, one after the other, plain
// tensor entries.  The planned layout is the library's own (two-site: fused per middle label, entries
// multiplied by sqrt(2 j_b + 1); one-site: identical to the interchange format).
static void ensure_io(fh_ctx* ctx) {
  Plan& P = ctx->plan;
  if (P.io_ready) return;
  std::vector<CopyBlk> imp(P.vec.keys.size()), exp_(P.vec.keys.size());
  int64_t canon = 0;
  for (size_t i = 0; i < P.vec.keys.size(); ++i) {
    const double w = P.nsite == 2 ? std::sqrt((double)(P.vec.keys[i][7] + 1)) : 1.0;
    CopyBlk b;
    b.rows = P.vec.rows[i];
    b.cols = P.vec.cols[i];
    b.transpose_dst = 0;
    b.pad = 0;
    b.src_off = canon;
    b.dst_off = P.vec.off[i];
    b.ld_src = P.vec.cols[i];
    b.ld_dst = P.vec.ld[i];
    b.scale = w;
    imp[i] = b;
    b.src_off = P.vec.off[i];
    b.dst_off = canon;
    b.ld_src = P.vec.ld[i];
    b.ld_dst = P.vec.cols[i];
    b.scale = 1.0 / w;
    exp_[i] = b;
    canon += (int64_t)P.vec.rows[i] * P.vec.cols[i];
  }
  FH_REQUIRE(canon == P.vec.nelem, FH_ESTATE, "planned layout and interchange format differ in size");
  P.n_io = (int)imp.size();
  P.io_pool.reset();
  P.io_pool.reserve(2 * imp.size() * sizeof(CopyBlk) + 4096, ctx->stream);
  P.d_import = upload(P.io_pool, imp, ctx->stream);
  P.d_export = upload(P.io_pool, exp_, ctx->stream);
  FH_CUDA(cudaStreamSynchronize(ctx->stream));  // imp / exp_ are stack-owned
  P.io_ready = true;
}
void fh::vec_import(fh_ctx* ctx, const cplx* blocks, cplx* vec) {
  FH_REQUIRE(ctx->plan.valid, FH_ESTATE, "heff_import: no plan (call heff_plan first)");
  ensure_io(ctx);
  launch_copy_blocks(ctx->plan.d_import, ctx->plan.n_io, blocks, vec, ctx->stream, &ctx->launches);
  FH_CUDA(cudaGetLastError());
}
void fh::vec_export(fh_ctx* ctx, const cplx* vec, cplx* blocks) {
  FH_REQUIRE(ctx->plan.valid, FH_ESTATE, "heff_export: no plan (call heff_plan first)");
  ensure_io(ctx);
  launch_copy_blocks(ctx->plan.d_export, ctx->plan.n_io, vec, blocks, ctx->stream, &ctx->launches);
  FH_CUDA(cudaGetLastError());
}

// Split-precision apply (NEXT-3): the same two stages, task lists, operands and intermediate as the FP64 apply, the
// products taken as 3 x TF32 on the tcgen05 tensor cores (zgemm_tc.cu)
static void apply_heff_tc(fh_ctx* ctx, const cplx* theta, cplx* out) {
  Plan& P = ctx->plan;
  if (!P.tc_ready) {
    // tile lists of both stages, and the static operand of each stage (stage 1: the left environment as op(A),
    // stage 2: the right environment as op(B)) converted ONCE per plan into panel images that the kernel streams
    // with bulk copies; the operand that changes with every apply (theta, Z) is converted inside the kernel
    std::vector<TcTile> t1, t2;
    std::vector<int> cb1, cb2;
    std::vector<int64_t> img1, img2;
    std::vector<TcPackChunk> pc1, pc2;
    build_tc_tiles(P.st1, ctx->num_sms, t1, cb1);
    build_tc_tiles(P.st2, ctx->num_sms, t2, cb2);
    const int64_t b1 = build_tc_static(P.st1, true, img1, pc1), b2 = build_tc_static(P.st2, false, img2, pc2);
    P.tc_pool.reset();
    P.tc_pool.reserve((t1.size() + t2.size()) * sizeof(TcTile) + (img1.size() + img2.size()) * 8 + 8 * (size_t)ctx->num_sms + 2048 +
                          (pc1.size() + pc2.size()) * sizeof(TcPackChunk) + (size_t)(b1 + b2) + 8192,
                      ctx->stream);
    P.d_tc1 = upload(P.tc_pool, t1, ctx->stream);
    P.d_tc2 = upload(P.tc_pool, t2, ctx->stream);
    P.d_tc_cb1 = upload(P.tc_pool, cb1, ctx->stream);
    P.d_tc_cb2 = upload(P.tc_pool, cb2, ctx->stream);
    P.d_tc_img1 = upload(P.tc_pool, img1, ctx->stream);
    P.d_tc_img2 = upload(P.tc_pool, img2, ctx->stream);
    TcPackChunk* d_pc1 = upload(P.tc_pool, pc1, ctx->stream);
    TcPackChunk* d_pc2 = upload(P.tc_pool, pc2, ctx->stream);
    P.tc_images1 = (unsigned char*)P.tc_pool.take((size_t)b1 + 256);
    P.tc_images2 = (unsigned char*)P.tc_pool.take((size_t)b2 + 256);
    P.n_tc1 = (int)t1.size();
    P.n_tc2 = (int)t2.size();
    launch_tc_pack(d_pc1, (int)pc1.size(), P.Lptr, P.tc_images1, P.st1.opA != OPA_N, ctx->stream, &ctx->launches);
    launch_tc_pack(d_pc2, (int)pc2.size(), P.Rptr, P.tc_images2, 0, ctx->stream, &ctx->launches);
    FH_CUDA(cudaGetLastError());
    FH_CUDA(cudaStreamSynchronize(ctx->stream));  // the host vectors are stack-owned
    P.tc_ready = true;
  }
  cplx* Z = ctx->ptr(P.Z.base);
  launch_grouped_gemm_tc(P.d_tc1, P.d_tc_cb1, ctx->num_sms, P.n_tc1, P.st1.d_segs, P.st1.opA != OPA_N, P.Lptr, theta, Z, ctx->stream,
                         &ctx->launches, 1, P.d_tc_img1, P.tc_images1);
  launch_grouped_gemm_tc(P.d_tc2, P.d_tc_cb2, ctx->num_sms, P.n_tc2, P.st2.d_segs, P.st2.opA != OPA_N, Z, P.Rptr, out, ctx->stream,
                         &ctx->launches, 2, P.d_tc_img2, P.tc_images2);
  FH_CUDA(cudaGetLastError());
}

void fh::apply_heff(fh_ctx* ctx, const cplx* theta, cplx* out) {
  Plan& P = ctx->plan;
  FH_REQUIRE(P.valid, FH_ESTATE, "heff_apply: no plan (call heff_plan first)");
  if (ctx->opt_precision == 1 && P.nsite == 2) return apply_heff_tc(ctx, theta, out);
  cplx* Z = ctx->ptr(P.Z.base);
  // Which form: measured on the Gaussian and Table-S2 profiles the warp-specialised single
  // launch wins from about 1e7 padded DMMAs per apply upwards (chi ~ 5000 - 12000: +5 ... +10 %), ties above and
  // at chi = 4096, and loses below (its start-up is longer than that of 148 x 8 one-warp CTAs).
  const int64_t dmma = P.st1.dmma_padded + P.st2.dmma_padded;
  const bool use_ws = P.nsite == 2 && !P.pair.tiles.empty() &&
                      (ctx->opt_gemm_path == 2 || (ctx->opt_gemm_path == 0 && dmma >= WS_MIN_DMMA && dmma < WS_MAX_DMMA));
  if (use_ws) {
    ++P.ws_epoch;
    cplx* sc = P.ws_scratch >= 0 ? ctx->ptr(P.ws_scratch) : nullptr;
    launch_grouped_gemm_ws_pair(P.pair, P.Lptr, theta, Z, Z, P.Rptr, out, ctx->d_ws_counters, ctx->num_sms, sc,
                                P.d_ws_flags, P.d_ws_dep, P.ws_epoch, ctx->stream, &ctx->launches);
  } else if (P.nsite == 2 && !P.upair.units.empty() && ctx->opt_gemm_path == 3) {
    // warp units, both stages in one launch (per-output dependency counters); set before heff_plan.  Measured 0.1667 ms
    // against 0.1611 ms for two launches at chi = 4096, equal elsewhere: an option, not the default
    ++P.unit_epoch;
    launch_grouped_gemm_pair(P.upair, P.Lptr, theta, Z, Z, P.Rptr, out, P.d_unit_dep, P.unit_epoch, ctx->stream, &ctx->launches);
  } else {
    launch_grouped_gemm(P.st1, P.Lptr, theta, Z, ctx->stream, &ctx->launches, PDL_GEMM_FIRST);
    launch_grouped_gemm(P.st2, Z, P.Rptr, out, ctx->stream, &ctx->launches, PDL_GEMM_SECOND);
  }
  FH_CUDA(cudaGetLastError());
}

double2 fh::inner(fh_ctx* ctx, const cplx* x, const cplx* y) {
  Plan& P = ctx->plan;
  FH_REQUIRE(P.valid, FH_ESTATE, "inner: no plan");
  ctx->ensure_pinned(2);
  if (P.chunks.empty()) return make_double2(0, 0);
  launch_wdot(P.d_chunks, (int)P.chunks.size(), x, y, P.d_partial, P.d_result, ctx->stream, &ctx->launches);
  FH_CUDA(cudaMemcpyAsync(ctx->h_pinned, P.d_result, 2 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
  FH_CUDA(cudaStreamSynchronize(ctx->stream));
  return make_double2(ctx->h_pinned[0], ctx->h_pinned[1]);
}

// symmetric tridiagonal eigen-decomposition by cyclic Jacobi (m <= 32): T = Q diag(lam) Q^T
static void jacobi_eig(int n, std::vector<double>& Amat, std::vector<double>& Q) {
  Q.assign(n * n, 0.0);
  for (int i = 0; i < n; ++i) Q[i * n + i] = 1.0;
  for (int sweep = 0; sweep < 100; ++sweep) {
    double offd = 0.0;
    for (int i = 0; i < n; ++i)
      for (int j = i + 1; j < n; ++j) offd += Amat[i * n + j] * Amat[i * n + j];
    if (offd < 1e-300) break;
    for (int p = 0; p < n; ++p)
      for (int q = p + 1; q < n; ++q) {
        const double apq = Amat[p * n + q];
        if (std::fabs(apq) < 1e-300) continue;
        const double app = Amat[p * n + p], aqq = Amat[q * n + q];
        const double theta = (aqq - app) / (2.0 * apq);
        const double t = (theta >= 0 ? 1.0 : -1.0) / (std::fabs(theta) + std::sqrt(theta * theta + 1.0));
        const double c = 1.0 / std::sqrt(t * t + 1.0), s = t * c;
        for (int k = 0; k < n; ++k) {
          const double akp = Amat[k * n + p], akq = Amat[k * n + q];
          Amat[k * n + p] = c * akp - s * akq;
          Amat[k * n + q] = s * akp + c * akq;
        }
        for (int k = 0; k < n; ++k) {
          const double apk = Amat[p * n + k], aqk = Amat[q * n + k];
          Amat[p * n + k] = c * apk - s * aqk;
          Amat[q * n + k] = s * apk + c * aqk;
        }
        for (int k = 0; k < n; ++k) {
          const double qkp = Q[k * n + p], qkq = Q[k * n + q];
          Q[k * n + p] = c * qkp - s * qkq;
          Q[k * n + q] = s * qkp + c * qkq;
        }
      }
  }
}

// u = exp(-i tau T_k) e_1 for the k x k tridiagonal T_k(alpha, beta) through its symmetric eigendecomposition (H7)
static std::vector<cplx> tridiag_exp_col(const std::vector<double>& alpha, const std::vector<double>& beta, int k,
                                         double tau) {
  std::vector<double> T(k * k, 0.0), Q;
  for (int i = 0; i < k; ++i) {
    T[i * k + i] = alpha[i];
    if (i + 1 < k) T[i * k + i + 1] = T[(i + 1) * k + i] = beta[i];
  }
  jacobi_eig(k, T, Q);
  std::vector<cplx> u(k);
  for (int i = 0; i < k; ++i) {
    double re = 0.0, im = 0.0;
    for (int l = 0; l < k; ++l) {
      const double lam = T[l * k + l], wgt = Q[i * k + l] * Q[0 * k + l];
      re += wgt * std::cos(tau * lam);
      im -= wgt * std::sin(tau * lam);
    }
    u[i] = make_double2(re, im);
  }
  return u;
}

// theta <- exp(-i tau H_eff) theta (H6 + H7).  work holds (m+1) vectors of n elements.
// The recurrence keeps alpha_j, <w,w> and beta_j in device memory (P.d_scal): with a fixed Krylov
// dimension (adapt_tol <= 0) there is no host round trip inside the iteration -- one copy of the scalars
// at the end, then the m x m tridiagonal problem on the host.  After a happy breakdown (beta_j < tol) the
// remaining directions are zero vectors and the host truncates the Krylov space at j.
// adapt_tol > 0 (NEXT-2, reading A-15): the scalars are read back after every step and the process stops
// with k = j + 1 vectors as soon as |tau| beta_j |e_k^T exp(-i tau T_k) e_1| <= adapt_tol (the norm of the
// ODE residual of the Krylov approximation times the step); one stream synchronisation per step.
int fh::expm_lanczos(fh_ctx* ctx, cplx* theta, double tau, int m, double tol, cplx* V, double adapt_tol) {
  Plan& P = ctx->plan;
  const int64_t n = P.vec.nelem;
  FH_REQUIRE(m >= 1 && m <= 32, FH_EINVAL, "krylov_dim must be in [1, 32]");
  if (n == 0 || P.chunks.empty()) return 0;
  cudaStream_t s = ctx->stream;
  const int nch = (int)P.chunks.size();
  // device scalars: [0,1] <theta,theta>, then per j: a_raw_j = <u_j, H u_j> at 2 + 4j, <u_{j+1}, u_{j+1}> at 4 + 4j.
  // The Krylov vectors are kept unnormalised, u_j = b_j v_j with b_0 = 1 and b_j = beta_{j-1} (kernels.cu,
  // lanczos_update_kernel): alpha_j = a_raw_j / b_j^2, beta_j = sqrt(<u_{j+1}, u_{j+1}>), and the final linear
  // combination takes c_j / b_j.
  double* d_sc = P.d_scal;
  const int nsc = 2 + 4 * 32 + 32;
  ctx->ensure_pinned(nsc);
  auto fetch_scalars = [&]() {
    FH_CUDA(cudaMemcpyAsync(ctx->h_pinned, d_sc, nsc * sizeof(double), cudaMemcpyDeviceToHost, s));
    FH_CUDA(cudaStreamSynchronize(s));
    check_fact_status(ctx);  // status words of the factorisations enqueued before this exponential
  };
  // reciprocal of b_j as the kernel takes it (0 below tol) from the fetched scalars
  auto recip_b = [&](int j) {
    if (j == 0) return 1.0;
    const double b = std::sqrt(std::max(ctx->h_pinned[4 + 4 * (j - 1)], 0.0));
    return (b < tol || b == 0.0) ? 0.0 : 1.0 / b;
  };
  auto alpha_of = [&](int j) {
    const double f = recip_b(j);
    return ctx->h_pinned[2 + 4 * j] * f * f;
  };
  auto beta_of = [&](int j) { return std::sqrt(std::max(ctx->h_pinned[4 + 4 * j], 0.0)); };
  ctx->timer_begin(T_VEC);
  launch_wdot_fused(P.d_chunks, nch, theta, theta, P.d_partial, d_sc, P.d_counter, s, &ctx->launches);
  launch_scale_rsqrt_dev(n, d_sc, 0.0, theta, V, nullptr, s, &ctx->launches);
  ctx->vec_bytes += 64 * n;
  ctx->timer_end();
  std::vector<double> alpha, beta;
  int k = 0;  // > 0 once the adaptive rule (or a breakdown seen by it) has fixed the dimension
  for (int j = 0; j < m; ++j) {
    cplx* vj = V + (int64_t)j * n;
    cplx* w = V + (int64_t)(j + 1) * n;
    ctx->timer_begin(T_HEFF);
    apply_heff(ctx, vj, w);
    ctx->timer_end();
    ctx->timer_begin(T_VEC);
    launch_wdot_fused(P.d_chunks, nch, vj, w, P.d_partial, d_sc + 2 + 4 * j, P.d_counter, s, &ctx->launches);
    ctx->vec_bytes += (32 + (j > 0 ? 64 : 48)) * n;
    launch_lanczos_update(P.d_chunks, nch, d_sc + 2 + 4 * j, j > 0 ? d_sc + 4 + 4 * (j - 1) : nullptr,
                          j > 1 ? d_sc + 4 + 4 * (j - 2) : nullptr, tol, vj, j > 0 ? V + (int64_t)(j - 1) * n : nullptr, w,
                          P.d_partial, d_sc + 4 + 4 * j, P.d_counter, s, &ctx->launches);
    ctx->timer_end();
    if (adapt_tol > 0.0 && j < m - 1) {
      fetch_scalars();
      if (!(ctx->h_pinned[0] > 0.0)) return 0;  // zero vector
      alpha.push_back(alpha_of(j));
      const double bj = beta_of(j);
      if (bj < tol) {
        k = j + 1;
        break;
      }
      const std::vector<cplx> u = tridiag_exp_col(alpha, beta, j + 1, tau);
      const double est = std::fabs(tau) * bj * std::hypot(u[j].x, u[j].y);
      if (est <= adapt_tol) {
        k = j + 1;
        break;
      }
      beta.push_back(bj);
    }
  }
  if (k == 0) {
    fetch_scalars();
    alpha.clear();
    beta.clear();
    for (int j = 0; j < m; ++j) {
      alpha.push_back(alpha_of(j));
      k = j + 1;
      if (j == m - 1) break;
      const double bj = beta_of(j);
      if (bj < tol) break;
      beta.push_back(bj);
    }
  }
  const double nrm2 = ctx->h_pinned[0];
  if (!(nrm2 > 0.0)) return 0;  // zero vector: theta is untouched (V holds zeros)
  const double nrm = std::sqrt(nrm2);
  std::vector<cplx> c = tridiag_exp_col(alpha, beta, k, tau);
  for (int j = 0; j < k; ++j) {  // v_j = u_j / b_j
    const double g = nrm * recip_b(j);
    c[j] = make_double2(g * c[j].x, g * c[j].y);
  }
  ctx->timer_begin(T_VEC);
  launch_lincomb(n, k, c.data(), V, n, theta, s, &ctx->launches);
  ctx->vec_bytes += 16 * (int64_t)(k + 1) * n;
  ctx->timer_end();
  FH_CUDA(cudaGetLastError());
  ctx->krylov_calls += 1;
  ctx->krylov_vectors += k;
  return k;
}

// ============================================================================ environments
static void run_two_stage(fh_ctx* ctx, Stage& st1, Stage& st2, BlockTensor& mid, const cplx* A1, const cplx* B1,
                          const cplx* A2_or_null, const cplx* B2_or_null, cplx* out, bool mid_is_lhs2) {
  // stage 1: mid = op(A1) op(B1); stage 2: out = op(lhs2) op(rhs2) where one operand is `mid`
  ctx->alloc_tensor(mid);
  ctx->pool_aux.reserve(stage_bytes(st1) + stage_bytes(st2) + 4096, ctx->stream);
  upload_stage(ctx->pool_aux, st1, ctx->stream);
  upload_stage(ctx->pool_aux, st2, ctx->stream);
  cplx* pm = ctx->ptr(mid.base);
  launch_grouped_gemm(st1, A1, B1, pm, ctx->stream, &ctx->launches);
  if (mid_is_lhs2) launch_grouped_gemm(st2, pm, B2_or_null, out, ctx->stream, &ctx->launches);
  else launch_grouped_gemm(st2, A2_or_null, pm, out, ctx->stream, &ctx->launches);
  FH_CUDA(cudaGetLastError());
  ctx->free_tensor(mid);
}

static std::vector<int> env_sig(const BlockTensor& E, const BlockTensor& A, const fh_mpo* mpo) {
  std::vector<int> sig;
  sig_add(sig, E);
  sig_add(sig, A);
  sig_add(sig, mpo->t_h);
  sig_add(sig, mpo->U);
  return sig;
}
static bool env_from_cache(fh_mps* mps, int kind, int site, const BlockTensor& E, const BlockTensor& A,
                           const fh_mpo* mpo, BlockTensor& mid, BlockTensor& out, Stage& st1, Stage& st2) {
  if (!mps->cache.enabled) return false;
  const PlanCacheEntry* e = mps->cache.find(kind, site, env_sig(E, A, mpo));
  if (!e) return false;
  mid = e->t0;
  out = e->t1;
  st1 = e->st1;
  st2 = e->st2;
  return true;
}
static void env_to_cache(fh_mps* mps, int kind, int site, const BlockTensor& E, const BlockTensor& A,
                         const fh_mpo* mpo, const BlockTensor& mid, const BlockTensor& out, const Stage& st1,
                         const Stage& st2) {
  if (!mps->cache.enabled) return;
  if (PlanCacheEntry* e = mps->cache.store(kind, site, env_sig(E, A, mpo))) {
    e->t0 = mid;
    e->t1 = out;
    e->st1 = st1;
    e->st2 = st2;
    mps->cache.account(e);
  }
}

void fh::do_env_update_left(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, int site) {
  FH_REQUIRE(site >= 0 && site < mps->L, FH_EINVAL, "env_update_left: site out of range");
  BlockTensor& Le = mps->Lenv[site];
  BlockTensor& A = mps->A[site];
  FH_REQUIRE(Le.base >= 0 && A.base >= 0, FH_ESTATE, "env_update_left: L_site or A_site missing");
  BlockTensor X, out;
  Stage st1, st2;
  if (!env_from_cache(mps, PC_ENVL, site, Le, A, mpo, X, out, st1, st2)) {
    emit_env_left(Le, A, mpo->site[site & 1], X, out, st1, st2);
    env_to_cache(mps, PC_ENVL, site, Le, A, mpo, X, out, st1, st2);
  }
  ctx->free_tensor(mps->Lenv[site + 1]);
  ctx->alloc_tensor(out);
  ctx->timer_begin(T_ENV);
  run_two_stage(ctx, st1, st2, X, ctx->ptr(Le.base), ctx->ptr(A.base), ctx->ptr(A.base), nullptr,
                ctx->ptr(out.base), false);
  ctx->timer_end();
  mps->Lenv[site + 1] = out;
}

void fh::do_env_update_right(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, int site) {
  FH_REQUIRE(site >= 0 && site < mps->L, FH_EINVAL, "env_update_right: site out of range");
  BlockTensor& Re = mps->Renv[site + 1];
  BlockTensor& A = mps->A[site];
  FH_REQUIRE(Re.base >= 0 && A.base >= 0, FH_ESTATE, "env_update_right: R_{site+1} or A_site missing");
  BlockTensor Y, out;
  Stage st1, st2;
  if (!env_from_cache(mps, PC_ENVR, site, Re, A, mpo, Y, out, st1, st2)) {
    emit_env_right(Re, A, mpo->site[site & 1], Y, out, st1, st2);
    env_to_cache(mps, PC_ENVR, site, Re, A, mpo, Y, out, st1, st2);
  }
  ctx->free_tensor(mps->Renv[site]);
  ctx->alloc_tensor(out);
  ctx->timer_begin(T_ENV);
  run_two_stage(ctx, st1, st2, Y, ctx->ptr(A.base), ctx->ptr(Re.base), nullptr, ctx->ptr(A.base),
                ctx->ptr(out.base), true);
  ctx->timer_end();
  mps->Renv[site] = out;
}

// ============================================================================ C ABI
#define FH_TRY(ctxptr, ...)                    \
  try {                                        \
    fh::SymScope sym_scope__((ctxptr) ? (ctxptr)->sym : nullptr); \
    __VA_ARGS__;                               \
    return FH_OK;                              \
  } catch (const fh::FhError& e) {             \
    if (ctxptr) (ctxptr)->err = e.what();      \
    return e.code;                             \
  } catch (const std::exception& e) {          \
    if (ctxptr) (ctxptr)->err = e.what();      \
    return FH_EINVAL;                          \
  }

// message of the last failed fh_ctx_create of this thread (there is no context to hold it): fh_last_error(NULL)
static thread_local std::string g_create_error = "null context";

extern "C" {

int fh_ctx_create(fh_ctx** out, void* cuda_stream, void* arena_dev, size_t arena_bytes) {
  if (!out || arena_bytes < (1u << 20)) return FH_EINVAL;
  fh_ctx* c = new fh_ctx();
  try {
    int ndev = 0;
    FH_CUDA(cudaGetDeviceCount(&ndev));
    FH_REQUIRE(ndev > 0, FH_ECUDA, "no CUDA device");
    c->stream = (cudaStream_t)cuda_stream;
    FH_CUDA(cudaGetDevice(&c->device));
    if (arena_dev) {
      c->arena = (cplx*)arena_dev;
    } else {
      FH_CUDA(cudaMalloc((void**)&c->arena, arena_bytes));
      c->own_arena = true;
    }
    c->alloc.init((int64_t)(arena_bytes / sizeof(cplx)));
    c->ensure_pinned(4096);
    FH_CUDA(cudaMalloc((void**)&c->d_ws_counters, 64));
    FH_CUDA(cudaMemset(c->d_ws_counters, 0, 64));
    {
      cudaDeviceProp prop;
      FH_CUDA(cudaGetDeviceProperties(&prop, c->device));
      c->num_sms = prop.multiProcessorCount;
    }
  } catch (const std::exception& e) {
    g_create_error = std::string("fh_ctx_create: ") + e.what();
    delete c;
    return FH_ECUDA;
  }
  *out = c;
  return FH_OK;
}

void fh_ctx_destroy(fh_ctx* c) {
  if (!c) return;
  fh::prefetch_cancel(c);
  cudaStreamSynchronize(c->stream);
  for (auto& sp : c->spans) {
    cudaEventDestroy(sp.a);
    cudaEventDestroy(sp.b);
  }
  for (auto e : c->ev_free) cudaEventDestroy(e);
  c->plan.pool.destroy();
  c->plan.io_pool.destroy();
  c->plan.tc_pool.destroy();
  if (c->d_ws_counters) cudaFree(c->d_ws_counters);
  if (c->d_fact_status) cudaFree(c->d_fact_status);
  if (c->h_fact_status) cudaFreeHost(c->h_fact_status);
  c->pool_aux.destroy();
  c->pool_small.destroy();
  for (auto& w : c->svd_workers) {
    if (w.s) cudaStreamSynchronize(w.s);
    if (w.h) cusolverDnDestroy(w.h);
    if (w.params) cusolverDnDestroyParams(w.params);
    if (w.cb) cublasDestroy(w.cb);
    if (w.dwork) cudaFree(w.dwork);
    if (w.d_info) cudaFree(w.d_info);
    if (w.done) cudaEventDestroy(w.done);
    if (w.s) cudaStreamDestroy(w.s);
  }
  if (c->svd_fork) cudaEventDestroy(c->svd_fork);
  if (c->small_copied) cudaEventDestroy(c->small_copied);
  if (c->svd_side_done) cudaEventDestroy(c->svd_side_done);
  if (c->svd_side) cudaStreamDestroy(c->svd_side);
  if (c->h_pinned) cudaFreeHost(c->h_pinned);
  if (c->own_arena) cudaFree(c->arena);
  delete c;
}

const char* fh_last_error(const fh_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

int fh_set_option(fh_ctx* c, int key, int value) {
  if (!c) return FH_EINVAL;
  switch (key) {
    case FH_OPT_GEMM_PATH:
      if (value < 0 || value > 3) return FH_EINVAL;
      c->opt_gemm_path = value;
      return FH_OK;
    case FH_OPT_SVD_MID_MAXN:
      if (value < 0 || value > 256) return FH_EINVAL;
      c->opt_svd_mid_maxn = value;
      return FH_OK;
    case FH_OPT_SVD_SMALL_MAXN:
      if (value < 0 || value > 4096) return FH_EINVAL;
      c->opt_svd_small_maxn = value;
      return FH_OK;
    case FH_OPT_SVD_GRAM_MINN:
      if (value < 0 || value > 65536) return FH_EINVAL;
      c->opt_svd_gram_minn = value;
      return FH_OK;
    case FH_OPT_SVD_GRAM_BATCH_MAXN:
      if (value < 0 || value > 65536) return FH_EINVAL;
      c->opt_svd_gram_batch_maxn = value;
      return FH_OK;
    case FH_OPT_PRECISION:
      if (value < 0 || value > 1) return FH_EINVAL;
      c->opt_precision = (int)value;
      return FH_OK;
    case FH_OPT_SYMMETRY:
      if (value < 0 || value > 1) return FH_EINVAL;
      c->sym = value == 1 ? &SYM_U1U1 : &SYM_SU2;
      return FH_OK;
    case FH_OPT_SVD_THREADS:
      if (value < 1 || value > 12) return FH_EINVAL;
      c->opt_svd_threads = value;
      return FH_OK;
    default:
      return FH_EINVAL;
  }
}

int fh_arena_stats(const fh_ctx* c, size_t* used, size_t* peak) {
  if (!c) return FH_EINVAL;
  if (used) *used = (size_t)c->alloc.used * sizeof(cplx);
  if (peak) *peak = (size_t)c->alloc.peak * sizeof(cplx);
  return FH_OK;
}

int fh_mpo_build(fh_ctx* ctx, int L, double t_h, double U, fh_mpo** out) {
  FH_TRY(ctx, {
    FH_REQUIRE(out != nullptr, FH_EINVAL, "fh_mpo_build: out is NULL");
    FH_REQUIRE(L >= 2 && L <= 4096 && L % 2 == 0, FH_EINVAL, "fh_mpo_build: L must be even, 2 <= L <= 4096");
    fh_mpo* m = new fh_mpo();
    m->sym = ctx->sym;
    m->L = L;
    m->t_h = t_h;
    m->U = U;
    mpo_site_table(0, t_h, U, m->site[0]);
    mpo_site_table(1, t_h, U, m->site[1]);
    *out = m;
  })
}
void fh_mpo_destroy(fh_mpo* m) { delete m; }

int fh_mpo_get_site(const fh_mpo* mpo, int site, double* val, int32_t* rank2) {
  if (!mpo || site < 0 || site >= mpo->L) return FH_EINVAL;
  const MpoSite& W = mpo->site[site & 1];
  if (val) std::memcpy(val, W.val, sizeof(W.val));
  if (rank2)
    for (int a = 0; a < MAX_NW; ++a)
      for (int b = 0; b < MAX_NW; ++b) rank2[a * MAX_NW + b] = W.rank2[a][b];
  return FH_OK;
}

static void set_boundaries(fh_ctx* ctx, fh_mps* m) {
  // L_0[(0,0),S,(0,0)] = 1, R_L[(0,0),F,(0,0)] = 1 (F-4)
  const cplx one = make_double2(1.0, 0.0);
  for (int which = 0; which < 2; ++which) {
    BlockTensor& E = which == 0 ? m->Lenv[0] : m->Renv[m->L];
    ctx->free_tensor(E);
    E.clear();
    E.nlab = 5;
    E.add(key_env(Sector{0, 0}, which == 0 ? 0 : sym().nw - 1, Sector{0, 0}), 1, 1);
    E.finalize();
    ctx->alloc_tensor(E);
    FH_CUDA(cudaMemcpyAsync(ctx->ptr(E.base), &one, sizeof(cplx), cudaMemcpyHostToDevice, ctx->stream));
  }
}

int mps_create(fh_ctx* ctx, int L, fh_mps** out) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && out, FH_EINVAL, "mps_create: NULL argument");
    FH_REQUIRE(L >= 2 && L <= 4096 && L % 2 == 0, FH_EINVAL, "mps_create: L must be even, 2 <= L <= 4096");
    fh_mps* m = new fh_mps();
    m->sym = ctx->sym;
    m->L = L;
    m->bond.resize(L + 1);
    m->A.resize(L);
    m->Lenv.resize(L + 1);
    m->Renv.resize(L + 1);
    m->sval.resize(L + 1);
    m->bond[0].sec = {Sector{0, 0}};
    m->bond[0].d = {1};
    m->bond[L] = m->bond[0];
    set_boundaries(ctx, m);
    *out = m;
  })
}

void mps_destroy(fh_ctx* ctx, fh_mps* m) {
  if (!m) return;
  if (ctx) {
    for (auto& t : m->A) ctx->free_tensor(t);
    for (auto& t : m->Lenv) ctx->free_tensor(t);
    for (auto& t : m->Renv) ctx->free_tensor(t);
  }
  delete m;
}

int mps_init_neel(fh_ctx* ctx, const fh_mpo* mpo, int L, fh_mps** out) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && mpo && out, FH_EINVAL, "mps_init_neel: NULL argument");
    FH_REQUIRE(mpo->L == L, FH_EINVAL, "mps_init_neel: L differs from the MPO's");
    fh_mps* m = nullptr;
    int rc = mps_create(ctx, L, &m);
    if (rc != FH_OK) throw FhError(rc, ctx->err);
    const cplx one = make_double2(1.0, 0.0);
    int q = 0;
    for (int i = 0; i < L; ++i) {
      const int up = sym().id == 1 ? 1 : 0;  // index of |up> among the site multiplets; |dn> follows it
      const int s = (i % 2 == 0) ? up : up + 1;
      const int qn = q + SITE_Q[s];
      m->bond[i + 1].sec = {Sector{qn, 0}};
      m->bond[i + 1].d = {1};
      BlockTensor& A = m->A[i];
      A.clear();
      A.nlab = 5;
      A.add(key_site(Sector{q, 0}, s, Sector{qn, 0}), 1, 1);
      A.finalize();
      ctx->alloc_tensor(A);
      FH_CUDA(cudaMemcpyAsync(ctx->ptr(A.base), &one, sizeof(cplx), cudaMemcpyHostToDevice, ctx->stream));
      q = qn;
    }
    for (int i = L - 1; i >= 1; --i) do_env_update_right(ctx, mpo, m, i);
    *out = m;
  })
}

// ---- checkpoint / resume: bond tables + site tensors of a state whose centre is on site 0
namespace {
struct FileCloser {
  FILE* f;
  ~FileCloser() { if (f) std::fclose(f); }
};
const char MPS_MAGIC[8] = {'F', 'H', 'M', 'P', 'S', '0', '1', 0};
}  // namespace

int mps_save(fh_ctx* ctx, const fh_mps* mps, const char* path) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && mps && path, FH_EINVAL, "mps_save: NULL argument");
    for (int i = 0; i < mps->L; ++i) FH_REQUIRE(mps->A[i].base >= 0, FH_ESTATE, "mps_save: site tensor missing");
    // written to path + ".tmp" and renamed once everything is on disk: a failed save never leaves a
    // truncated file under the final name
    const std::string tmp = std::string(path) + ".tmp";
    FileCloser fc{std::fopen(tmp.c_str(), "wb")};
    FH_REQUIRE(fc.f, FH_EINVAL, std::string("mps_save: cannot open ") + tmp);
    auto put = [&](const void* p, size_t n) {
      FH_REQUIRE(std::fwrite(p, 1, n, fc.f) == n, FH_EINVAL, "mps_save: short write");
    };
    const int32_t head[2] = {mps->L, mps->saturated ? 1 : 0};
    put(MPS_MAGIC, 8);
    put(head, sizeof(head));
    for (int k = 0; k <= mps->L; ++k) {
      const Bond& b = mps->bond[k];
      const int32_t n = (int32_t)b.sec.size();
      put(&n, 4);
      for (int32_t i = 0; i < n; ++i) {
        const int32_t rec[3] = {b.sec[i].q, b.sec[i].tj, b.d[i]};
        put(rec, sizeof(rec));
      }
    }
    std::vector<cplx> host;
    for (int i = 0; i < mps->L; ++i) {
      const BlockTensor& t = mps->A[i];
      BlockTensor ref;
      layout_site(mps->bond[i], mps->bond[i + 1], ref);
      FH_REQUIRE(ref.nelem == t.nelem && ref.keys == t.keys, FH_ESTATE, "mps_save: site tensor not in the bond tables' layout");
      host.resize((size_t)t.nelem);
      FH_CUDA(cudaMemcpyAsync(host.data(), ctx->ptr(t.base), t.nelem * sizeof(cplx), cudaMemcpyDeviceToHost, ctx->stream));
      FH_CUDA(cudaStreamSynchronize(ctx->stream));
      const int64_t ne = t.nelem;
      put(&ne, 8);
      put(host.data(), (size_t)ne * sizeof(cplx));
    }
    const bool flushed = std::fflush(fc.f) == 0;
    const bool closed = std::fclose(fc.f) == 0;
    fc.f = nullptr;
    if (!flushed || !closed || std::rename(tmp.c_str(), path) != 0) {
      std::remove(tmp.c_str());
      throw FhError(FH_EINVAL, std::string("mps_save: could not complete ") + path);
    }
  })
}

int mps_load(fh_ctx* ctx, const fh_mpo* mpo, const char* path, fh_mps** out) {
  fh_mps* m = nullptr;
  const int rc = [&]() -> int {
    FH_TRY(ctx, {
      FH_REQUIRE(ctx && mpo && path && out, FH_EINVAL, "mps_load: NULL argument");
      FileCloser fc{std::fopen(path, "rb")};
      FH_REQUIRE(fc.f, FH_EINVAL, std::string("mps_load: cannot open ") + path);
      auto get = [&](void* p, size_t n) {
        FH_REQUIRE(std::fread(p, 1, n, fc.f) == n, FH_EINVAL, "mps_load: truncated file");
      };
      char magic[8];
      int32_t head[2];
      get(magic, 8);
      FH_REQUIRE(std::memcmp(magic, MPS_MAGIC, 8) == 0, FH_EINVAL, "mps_load: not an fh_mps checkpoint");
      get(head, sizeof(head));
      FH_REQUIRE(head[0] == mpo->L, FH_EINVAL, "mps_load: chain length differs from the MPO's");
      int rc2 = mps_create(ctx, head[0], &m);
      if (rc2 != FH_OK) throw FhError(rc2, ctx->err);
      m->saturated = head[1] != 0;
      for (int k = 0; k <= m->L; ++k) {
        int32_t n = 0;
        get(&n, 4);
        FH_REQUIRE(n >= 1 && n <= (1 << 20), FH_EINVAL, "mps_load: bad sector count");
        Bond b;
        for (int32_t i = 0; i < n; ++i) {
          int32_t rec[3];
          get(rec, sizeof(rec));
          FH_REQUIRE(rec[1] >= 0 && rec[1] <= 250 && rec[2] >= 1 && rec[0] >= -8000 && rec[0] <= 8000, FH_EINVAL,
                     "mps_load: bad sector record");
          if (i > 0) FH_REQUIRE(b.sec.back() < Sector({rec[0], rec[1]}), FH_EINVAL, "mps_load: sector labels not sorted");
          b.sec.push_back(Sector{rec[0], rec[1]});
          b.d.push_back(rec[2]);
        }
        m->bond[k] = b;
      }
      std::vector<cplx> host;
      for (int i = 0; i < m->L; ++i) {
        BlockTensor t;
        layout_site(m->bond[i], m->bond[i + 1], t);
        int64_t ne = 0;
        get(&ne, 8);
        FH_REQUIRE(ne == t.nelem, FH_EINVAL, "mps_load: site tensor size does not match the bond tables");
        host.resize((size_t)ne);
        get(host.data(), (size_t)ne * sizeof(cplx));
        ctx->alloc_tensor(t);
        m->A[i] = t;
        FH_CUDA(cudaMemcpyAsync(ctx->ptr(t.base), host.data(), ne * sizeof(cplx), cudaMemcpyHostToDevice, ctx->stream));
        FH_CUDA(cudaStreamSynchronize(ctx->stream));
      }
      for (int i = m->L - 1; i >= 1; --i) do_env_update_right(ctx, mpo, m, i);
      *out = m;
    })
  }();
  if (rc != FH_OK && m) mps_destroy(ctx, m);
  return rc;
}

int mps_set_bond(fh_ctx* ctx, fh_mps* mps, int bond, int n, const int32_t* q, const int32_t* tj, const int32_t* d) {
  FH_TRY(ctx, {
    FH_REQUIRE(mps && bond >= 0 && bond <= mps->L && n >= 1, FH_EINVAL, "mps_set_bond: bad argument");
    Bond b;
    for (int i = 0; i < n; ++i) {
      FH_REQUIRE(tj[i] >= 0 && tj[i] <= 250 && d[i] >= 1, FH_EINVAL, "mps_set_bond: 0 <= tj <= 250 and d >= 1 required");
      FH_REQUIRE(q[i] >= -8000 && q[i] <= 8000, FH_EINVAL, "mps_set_bond: |q| <= 8000 required");
      if (sym().id == 0)
        FH_REQUIRE(((q[i] + tj[i] - bond) & 1) == 0, FH_EINVAL, "mps_set_bond: parity rule q + 2j = bond (mod 2) violated");
      else
        FH_REQUIRE(tj[i] == 0, FH_EINVAL, "mps_set_bond: U(1) x U(1) labels have tj = 0");
      if (i > 0) FH_REQUIRE(Sector({q[i - 1], tj[i - 1]}) < Sector({q[i], tj[i]}), FH_EINVAL, "mps_set_bond: labels must be sorted by (q, tj) and distinct");
      b.sec.push_back(Sector{q[i], tj[i]});
      b.d.push_back(d[i]);
    }
    if (bond == 0 || bond == mps->L)
      FH_REQUIRE(n == 1 && q[0] == 0 && tj[0] == 0 && d[0] == 1, FH_EINVAL, "mps_set_bond: boundary bonds are the single sector (0,0), d=1");
    mps->bond[bond] = b;
  })
}

int mps_get_bond(const fh_mps* mps, int bond, int* n, int32_t* q, int32_t* tj, int32_t* d) {
  if (!mps || bond < 0 || bond > mps->L || !n) return FH_EINVAL;
  const Bond& b = mps->bond[bond];
  *n = (int)b.sec.size();
  for (size_t i = 0; i < b.sec.size(); ++i) {
    if (q) q[i] = b.sec[i].q;
    if (tj) tj[i] = b.sec[i].tj;
    if (d) d[i] = b.d[i];
  }
  return FH_OK;
}

static void export_layout(const BlockTensor& t, int nlab, int* nblk, int64_t* nelem, int32_t* labels, int32_t* dims) {
  if (nblk) *nblk = (int)t.keys.size();
  if (nelem) *nelem = t.nelem;
  for (size_t i = 0; i < t.keys.size(); ++i) {
    if (labels)
      for (int l = 0; l < nlab; ++l) labels[i * nlab + l] = t.keys[i][l];
    if (dims) {
      dims[2 * i] = t.rows[i];
      dims[2 * i + 1] = t.cols[i];
    }
  }
}

int mps_site_layout(const fh_mps* mps, int site, int* nblk, int64_t* nelem, int32_t* labels, int32_t* dims) {
  fh::SymScope sym_scope(mps ? mps->sym : nullptr);
  if (!mps || site < 0 || site >= mps->L) return FH_EINVAL;
  if (mps->A[site].base >= 0 || !mps->A[site].keys.empty()) {
    export_layout(mps->A[site], 5, nblk, nelem, labels, dims);
  } else {
    BlockTensor t;
    layout_site(mps->bond[site], mps->bond[site + 1], t);
    export_layout(t, 5, nblk, nelem, labels, dims);
  }
  return FH_OK;
}

int mps_set_site(fh_ctx* ctx, fh_mps* mps, int site, const void* data, int is_dev) {
  FH_TRY(ctx, {
    FH_REQUIRE(mps && site >= 0 && site < mps->L && data, FH_EINVAL, "mps_set_site: bad argument");
    BlockTensor t;
    layout_site(mps->bond[site], mps->bond[site + 1], t);
    ctx->free_tensor(mps->A[site]);
    ctx->alloc_tensor(t);
    FH_CUDA(cudaMemcpyAsync(ctx->ptr(t.base), data, t.nelem * sizeof(cplx),
                            is_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, ctx->stream));
    if (!is_dev) FH_CUDA(cudaStreamSynchronize(ctx->stream));
    mps->A[site] = t;
  })
}

int mps_get_site(fh_ctx* ctx, const fh_mps* mps, int site, void* data, int64_t capacity, int is_dev) {
  FH_TRY(ctx, {
    FH_REQUIRE(mps && site >= 0 && site < mps->L && data, FH_EINVAL, "mps_get_site: bad argument");
    const BlockTensor& t = mps->A[site];
    FH_REQUIRE(t.base >= 0, FH_ESTATE, "mps_get_site: site tensor not set");
    FH_REQUIRE(capacity >= t.nelem, FH_EINVAL, "mps_get_site: buffer smaller than the site tensor (mps_site_layout gives nelem)");
    FH_CUDA(cudaMemcpyAsync(data, ctx->ptr(t.base), t.nelem * sizeof(cplx),
                            is_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream));
    FH_CUDA(cudaStreamSynchronize(ctx->stream));
  })
}

int mps_get_svals(const fh_mps* mps, int bond, int* n, double* s) {
  if (!mps || bond < 0 || bond > mps->L || !n) return FH_EINVAL;
  const std::vector<double>& v = mps->sval[bond];
  *n = (int)v.size();
  if (s) std::memcpy(s, v.data(), v.size() * sizeof(double));
  return FH_OK;
}

int mps_drop_site(fh_ctx* ctx, fh_mps* mps, int site) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && mps && site >= 0 && site < mps->L, FH_EINVAL, "mps_drop_site: bad argument");
    ctx->free_tensor(mps->A[site]);
    mps->A[site].clear();
  })
}

int env_update_left(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, int site) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && mpo && mps, FH_EINVAL, "env_update_left: NULL argument");
    do_env_update_left(ctx, mpo, mps, site);
  })
}
int env_update_right(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, int site) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && mpo && mps, FH_EINVAL, "env_update_right: NULL argument");
    do_env_update_right(ctx, mpo, mps, site);
  })
}

int env_layout(const fh_mps* mps, int which, int bond, int* nblk, int64_t* nelem, int32_t* labels, int32_t* dims) {
  if (!mps || bond < 0 || bond > mps->L || (which != 0 && which != 1)) return FH_EINVAL;
  const BlockTensor& t = which == 0 ? mps->Lenv[bond] : mps->Renv[bond];
  if (t.base < 0) return FH_ESTATE;
  export_layout(t, 5, nblk, nelem, labels, dims);
  return FH_OK;
}

int env_get(fh_ctx* ctx, const fh_mps* mps, int which, int bond, void* data, int64_t capacity, int is_dev) {
  FH_TRY(ctx, {
    FH_REQUIRE(mps && bond >= 0 && bond <= mps->L && data && (which == 0 || which == 1), FH_EINVAL, "env_get: bad argument");
    const BlockTensor& t = which == 0 ? mps->Lenv[bond] : mps->Renv[bond];
    FH_REQUIRE(t.base >= 0, FH_ESTATE, "env_get: environment not built");
    FH_REQUIRE(capacity >= t.nelem, FH_EINVAL, "env_get: buffer smaller than the environment (env_layout gives nelem)");
    FH_CUDA(cudaMemcpyAsync(data, ctx->ptr(t.base), t.nelem * sizeof(cplx),
                            is_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream));
    FH_CUDA(cudaStreamSynchronize(ctx->stream));
  })
}

int env_set(fh_ctx* ctx, fh_mps* mps, int which, int bond, int nblk, const int32_t* labels, const void* data, int is_dev) {
  FH_TRY(ctx, {
    FH_REQUIRE(mps && bond >= 0 && bond <= mps->L && data && labels && nblk >= 1 && (which == 0 || which == 1), FH_EINVAL, "env_set: bad argument");
    const Bond& b = mps->bond[bond];
    BlockTensor t;
    t.nlab = 5;
    for (int i = 0; i < nblk; ++i) {
      const int32_t* l = labels + 5 * i;
      const Sector xp{l[0], l[1]}, x{l[3], l[4]};
      const int w = l[2];
      FH_REQUIRE(w >= 0 && w < sym().nw && b.find(xp) >= 0 && b.find(x) >= 0, FH_EINVAL, "env_set: label not in the bond table");
      FH_REQUIRE(xp.q == x.q + MPO_Q[w] && triangle(x.tj, MPO_TK[w], xp.tj), FH_EINVAL, "env_set: block violates the selection rule");
      const Key k = key_env(xp, w, x);
      if (i > 0) FH_REQUIRE(t.keys.back() < k, FH_EINVAL, "env_set: blocks must be in canonical order");
      t.add(k, b.dim(xp), b.dim(x));
    }
    t.finalize();
    BlockTensor& E = which == 0 ? mps->Lenv[bond] : mps->Renv[bond];
    ctx->free_tensor(E);
    ctx->alloc_tensor(t);
    FH_CUDA(cudaMemcpyAsync(ctx->ptr(t.base), data, t.nelem * sizeof(cplx),
                            is_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, ctx->stream));
    if (!is_dev) FH_CUDA(cudaStreamSynchronize(ctx->stream));
    E = t;
  })
}

int heff_plan(fh_ctx* ctx, const fh_mpo* mpo, const fh_mps* mps, int site, int nsite) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && mpo && mps, FH_EINVAL, "heff_plan: NULL argument");
    plan_heff(ctx, mpo, mps, site, nsite);
  })
}

int heff_layout(const fh_ctx* ctx, int* nblk, int64_t* nelem, int32_t* labels, int32_t* dims) {
  if (!ctx || !ctx->plan.valid) return FH_ESTATE;
  export_layout(ctx->plan.vec, ctx->plan.nsite == 2 ? 8 : 5, nblk, nelem, labels, dims);
  return FH_OK;
}

int heff_get_tasks(const fh_ctx* ctx, int stage, int* ntask, int* nout, int32_t* tuples, double* alpha) {
  if (!ctx || !ctx->plan.valid || (stage != 1 && stage != 2)) return FH_ESTATE;
  const Stage& st = stage == 1 ? ctx->plan.st1 : ctx->plan.st2;
  if (ntask) *ntask = (int)st.t_out.size();
  if (nout) *nout = (int)st.outs.size();
  for (size_t i = 0; i < st.t_out.size(); ++i) {
    if (tuples) {
      tuples[3 * i] = st.t_out[i];
      tuples[3 * i + 1] = st.t_lhs[i];
      tuples[3 * i + 2] = st.t_rhs[i];
    }
    if (alpha) alpha[i] = st.t_alpha[i];
  }
  return FH_OK;
}

int heff_apply(fh_ctx* ctx, const void* theta_dev, void* out_dev) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && theta_dev && out_dev, FH_EINVAL, "heff_apply: NULL argument");
    apply_heff(ctx, (const cplx*)theta_dev, (cplx*)out_dev);
  })
}

int heff_import(fh_ctx* ctx, const void* blocks_dev, void* vec_dev) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && blocks_dev && vec_dev && blocks_dev != vec_dev, FH_EINVAL, "heff_import: bad argument");
    vec_import(ctx, (const cplx*)blocks_dev, (cplx*)vec_dev);
  })
}

int heff_export(fh_ctx* ctx, const void* vec_dev, void* blocks_dev) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && blocks_dev && vec_dev && blocks_dev != vec_dev, FH_EINVAL, "heff_export: bad argument");
    vec_export(ctx, (const cplx*)vec_dev, (cplx*)blocks_dev);
  })
}

int heff_apply_host(fh_ctx* ctx, const void* theta_host, void* out_host) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && theta_host && out_host, FH_EINVAL, "heff_apply_host: NULL argument");
    FH_REQUIRE(ctx->plan.valid, FH_ESTATE, "heff_apply_host: no plan (call heff_plan first)");
    const int64_t n = ctx->plan.vec.nelem;
    const int64_t off = ctx->alloc.alloc(3 * n);
    try {
      cplx* io = ctx->ptr(off);
      cplx* din = io + n;
      cplx* dout = din + n;
      FH_CUDA(cudaMemcpyAsync(io, theta_host, n * sizeof(cplx), cudaMemcpyHostToDevice, ctx->stream));
      vec_import(ctx, io, din);
      apply_heff(ctx, din, dout);
      vec_export(ctx, dout, io);
      FH_CUDA(cudaMemcpyAsync(out_host, io, n * sizeof(cplx), cudaMemcpyDeviceToHost, ctx->stream));
      FH_CUDA(cudaStreamSynchronize(ctx->stream));
    } catch (...) {
      ctx->alloc.release(off, 3 * n);
      throw;
    }
    ctx->alloc.release(off, 3 * n);
  })
}

int64_t heff_flops(const fh_ctx* ctx) {
  if (!ctx || !ctx->plan.valid) return -1;
  return ctx->plan.st1.flops + ctx->plan.st2.flops;
}

int heff_inner(fh_ctx* ctx, const void* x_dev, const void* y_dev, double* result) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && x_dev && y_dev && result, FH_EINVAL, "heff_inner: NULL argument");
    const double2 r = inner(ctx, (const cplx*)x_dev, (const cplx*)y_dev);
    result[0] = r.x;
    result[1] = r.y;
  })
}

static int heff_expm_impl(fh_ctx* ctx, const void* theta_dev, void* out_dev, double tau, int krylov_dim,
                          double adapt_tol, int* k_used) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && theta_dev && out_dev, FH_EINVAL, "heff_expm: NULL argument");
    FH_REQUIRE(ctx->plan.valid, FH_ESTATE, "heff_expm: no plan");
    const int64_t n = ctx->plan.vec.nelem;
    const int64_t woff = ctx->alloc.alloc((int64_t)(krylov_dim + 1) * n);
    try {
      if (out_dev != theta_dev)
        FH_CUDA(cudaMemcpyAsync(out_dev, theta_dev, n * sizeof(cplx), cudaMemcpyDeviceToDevice, ctx->stream));
      const int k = expm_lanczos(ctx, (cplx*)out_dev, tau, krylov_dim, 1e-12, ctx->ptr(woff), adapt_tol);
      if (k_used) *k_used = k;
    } catch (...) {
      ctx->alloc.release(woff, (int64_t)(krylov_dim + 1) * n);
      throw;
    }
    ctx->alloc.release(woff, (int64_t)(krylov_dim + 1) * n);
  })
}

int heff_expm(fh_ctx* ctx, const void* theta_dev, void* out_dev, double tau, int krylov_dim) {
  return heff_expm_impl(ctx, theta_dev, out_dev, tau, krylov_dim, 0.0, nullptr);
}

int heff_expm_adaptive(fh_ctx* ctx, const void* theta_dev, void* out_dev, double tau, int krylov_dim,
                       double adapt_tol, int* k_used) {
  if (!(adapt_tol > 0.0)) {
    if (ctx) ctx->err = "heff_expm_adaptive: adapt_tol must be > 0";
    return FH_EINVAL;
  }
  return heff_expm_impl(ctx, theta_dev, out_dev, tau, krylov_dim, adapt_tol, k_used);
}

int fh_factorization_stats(const fh_ctx* ctx, int64_t counts[9]) {
  if (!ctx || !counts) return FH_EINVAL;
  counts[7] = ctx->svd_count[3];
  counts[8] = ctx->svd_gram_redone;
  counts[6] = ctx->svd_mid;
  counts[5] = ctx->qr_small;
  counts[0] = ctx->svd_small;
  counts[1] = ctx->svd_count[1];
  counts[2] = ctx->svd_count[0];
  counts[3] = ctx->svd_count[2];
  counts[4] = ctx->qr_count;
  return FH_OK;
}

int fh_plan_cache_stats(const fh_mps* mps, int64_t* hits, int64_t* misses, int64_t* host_bytes) {
  if (!mps) return FH_EINVAL;
  if (hits) *hits = mps->cache.hits;
  if (misses) *misses = mps->cache.misses;
  if (host_bytes) *host_bytes = (int64_t)mps->cache.bytes;
  return FH_OK;
}

int fh_plan_cache_limit(fh_mps* mps, int64_t max_host_bytes) {
  if (!mps || max_host_bytes < 0) return FH_EINVAL;
  mps->cache.clear();
  mps->cache.max_bytes = (size_t)max_host_bytes;
  return FH_OK;
}

int fh_krylov_stats(const fh_ctx* ctx, int64_t* n_exponentials, int64_t* n_vectors) {
  if (!ctx) return FH_EINVAL;
  if (n_exponentials) *n_exponentials = ctx->krylov_calls;
  if (n_vectors) *n_vectors = ctx->krylov_vectors;
  return FH_OK;
}

int tdvp2_sweep(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, double dt, const fh_params* p) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && mpo && mps && p, FH_EINVAL, "tdvp2_sweep: NULL argument");
    FH_REQUIRE(p->krylov_dim >= 2 && p->krylov_dim <= 32 && p->chi_max_full >= 1, FH_EINVAL, "tdvp2_sweep: bad parameters");
    sweep(ctx, mpo, mps, dt, p);
  })
}

int tdvp_sweep_auto(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, double dt, const fh_params* p, int* nsite_used) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && mpo && mps && p, FH_EINVAL, "tdvp_sweep_auto: NULL argument");
    FH_REQUIRE(p->krylov_dim >= 2 && p->krylov_dim <= 32 && p->chi_max_full >= 1, FH_EINVAL,
               "tdvp_sweep_auto: bad parameters");
    if (mps->saturated) {
      if (nsite_used) *nsite_used = 1;
      sweep1(ctx, mpo, mps, dt, p);
    } else {
      if (nsite_used) *nsite_used = 2;
      std::vector<int> before;
      for (const auto& b : mps->bond) before.push_back(b.chi_full());
      sweep(ctx, mpo, mps, dt, p);
      bool grew = false;
      for (size_t k = 0; k < mps->bond.size(); ++k) grew = grew || mps->bond[k].chi_full() > before[k];
      mps->saturated = !grew;
    }
  })
}

int tdvp1_sweep(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, double dt, const fh_params* p) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && mpo && mps && p, FH_EINVAL, "tdvp1_sweep: NULL argument");
    FH_REQUIRE(p->krylov_dim >= 2 && p->krylov_dim <= 32, FH_EINVAL, "tdvp1_sweep: bad parameters");
    sweep1(ctx, mpo, mps, dt, p);
  })
}

int tdvp2_last_stats(const fh_ctx* ctx, double* disc, int* chi_full, int* chi_su2, int* dmax) {
  if (!ctx) return FH_EINVAL;
  if (disc) *disc = ctx->stat_disc;
  if (chi_full) *chi_full = ctx->stat_chi;
  if (chi_su2) *chi_su2 = ctx->stat_su2;
  if (dmax) *dmax = ctx->stat_dmax;
  return FH_OK;
}

int measure_local(fh_ctx* ctx, const fh_mps* mps, double* n_i, double* sz_i, double* docc_i) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && mps && n_i && sz_i && docc_i, FH_EINVAL, "measure_local: NULL argument");
    measure_local_impl(ctx, mps, n_i, sz_i, docc_i);
  })
}

int measure_global(fh_ctx* ctx, const fh_mpo* mpo, const fh_mps* mps, double* norm2, double* energy) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && mpo && mps, FH_EINVAL, "measure_global: NULL argument");
    // full left contraction on a scratch copy of the left environments
    fh_mps tmp;
    tmp.L = mps->L;
    tmp.bond = mps->bond;
    tmp.A = mps->A;  // shares device storage (read only)
    tmp.Lenv.resize(mps->L + 1);
    tmp.Renv.resize(mps->L + 1);
    tmp.Lenv[0] = mps->Lenv[0];
    for (int i = 0; i < mps->L; ++i) {
      do_env_update_left(ctx, mpo, &tmp, i);
      if (i > 0) ctx->free_tensor(tmp.Lenv[i]);
    }
    BlockTensor& E = tmp.Lenv[mps->L];
    const int is = E.find(key_env(Sector{0, 0}, 0, Sector{0, 0})), ie = E.find(key_env(Sector{0, 0}, sym().nw - 1, Sector{0, 0}));
    std::vector<cplx> h(E.nelem);
    FH_CUDA(cudaMemcpyAsync(h.data(), ctx->ptr(E.base), E.nelem * sizeof(cplx), cudaMemcpyDeviceToHost, ctx->stream));
    FH_CUDA(cudaStreamSynchronize(ctx->stream));
    const double n2 = is >= 0 ? h[E.off[is]].x : 0.0;
    if (norm2) *norm2 = n2;
    if (energy) *energy = (ie >= 0 && n2 != 0.0) ? h[E.off[ie]].x / n2 : 0.0;
    ctx->free_tensor(E);
  })
}

int fh_get_timers(const fh_ctx* cctx, double* a, double* b, double* c, double* d, double* e) {
  fh_ctx* ctx = const_cast<fh_ctx*>(cctx);
  FH_TRY(ctx, {
    FH_REQUIRE(ctx != nullptr, FH_EINVAL, "fh_get_timers: NULL context");
    ctx->timers_resolve();
    if (a) *a = ctx->sec[T_HEFF];
    if (b) *b = ctx->sec[T_ENV];
    if (c) *c = ctx->sec[T_SVD];
    if (d) *d = ctx->sec[T_VEC];
    if (e) *e = ctx->sec[T_PACK];
  })
}
int fh_reset_timers(fh_ctx* ctx) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx != nullptr, FH_EINVAL, "fh_reset_timers: NULL context");
    ctx->timers_resolve();
    for (int i = 0; i < T_NCAT; ++i) ctx->sec[i] = 0.0;
    ctx->vec_bytes = ctx->pack_bytes = 0;
  })
}
int fh_get_traffic(const fh_ctx* ctx, int64_t* vec_bytes, int64_t* pack_bytes) {
  if (!ctx) return FH_EINVAL;
  if (vec_bytes) *vec_bytes = ctx->vec_bytes;
  if (pack_bytes) *pack_bytes = ctx->pack_bytes;
  return FH_OK;
}
int fh_enable_timers(fh_ctx* ctx, int on) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx != nullptr, FH_EINVAL, "fh_enable_timers: NULL context");
    ctx->timers_resolve();
    ctx->timers_on = on != 0;
  })
}
int64_t fh_launch_count(const fh_ctx* ctx) { return ctx ? ctx->launches : -1; }

int fh_cublas_gemm_seconds(fh_ctx* ctx, int n, int is_complex, int reps, double* seconds) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && n > 0 && reps > 0 && seconds, FH_EINVAL, "fh_cublas_gemm_seconds: bad argument");
    cublasHandle_t h;
    FH_REQUIRE(cublasCreate(&h) == CUBLAS_STATUS_SUCCESS, FH_ECUDA, "cublasCreate failed");
    cublasSetStream(h, ctx->stream);
    const size_t el = is_complex ? 16 : 8;
    void *A, *B, *C;
    FH_CUDA(cudaMalloc(&A, el * n * n));
    FH_CUDA(cudaMalloc(&B, el * n * n));
    FH_CUDA(cudaMalloc(&C, el * n * n));
    FH_CUDA(cudaMemsetAsync(A, 0x3c, el * n * n, ctx->stream));
    FH_CUDA(cudaMemsetAsync(B, 0x3c, el * n * n, ctx->stream));
    cudaEvent_t e0, e1;
    FH_CUDA(cudaEventCreate(&e0));
    FH_CUDA(cudaEventCreate(&e1));
    const double one = 1.0, zero = 0.0;
    const cuDoubleComplex zone = make_cuDoubleComplex(1, 0), zzero = make_cuDoubleComplex(0, 0);
    for (int it = -2; it < reps; ++it) {
      if (it == 0) FH_CUDA(cudaEventRecord(e0, ctx->stream));
      if (is_complex)
        cublasZgemm(h, CUBLAS_OP_N, CUBLAS_OP_N, n, n, n, &zone, (cuDoubleComplex*)A, n, (cuDoubleComplex*)B, n, &zzero, (cuDoubleComplex*)C, n);
      else
        cublasDgemm(h, CUBLAS_OP_N, CUBLAS_OP_N, n, n, n, &one, (double*)A, n, (double*)B, n, &zero, (double*)C, n);
    }
    FH_CUDA(cudaEventRecord(e1, ctx->stream));
    FH_CUDA(cudaEventSynchronize(e1));
    float ms = 0;
    FH_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    *seconds = ms * 1e-3 / reps;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(A);
    cudaFree(B);
    cudaFree(C);
    cublasDestroy(h);
  })
}

int fh_dmma_peak_tflops(fh_ctx* ctx, int reps, double* tflops) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && reps > 0 && tflops, FH_EINVAL, "fh_dmma_peak_tflops: bad argument");
    double* scratch = nullptr;
    FH_CUDA(cudaMalloc((void**)&scratch, (size_t)148 * 4 * 256 * sizeof(double)));
    cudaEvent_t e0, e1;
    FH_CUDA(cudaEventCreate(&e0));
    FH_CUDA(cudaEventCreate(&e1));
    const double fl = fh::launch_dmma_peak(scratch, ctx->stream, &ctx->launches);  // warm-up
    FH_CUDA(cudaEventRecord(e0, ctx->stream));
    for (int r = 0; r < reps; ++r) fh::launch_dmma_peak(scratch, ctx->stream, &ctx->launches);
    FH_CUDA(cudaEventRecord(e1, ctx->stream));
    FH_CUDA(cudaEventSynchronize(e1));
    float ms = 0;
    FH_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    *tflops = fl * reps / (ms * 1e-3) * 1e-12;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(scratch);
  })
}

int fh_vec_kernels_gbs(fh_ctx* ctx, int64_t n, int m, int reps, double* gbs) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && gbs && n >= 65536 && m >= 1 && m <= 32 && reps > 0, FH_EINVAL, "fh_vec_kernels_gbs: bad argument");
    const int64_t off = ctx->alloc.alloc((int64_t)(m + 3) * n);
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    try {
      cudaStream_t s = ctx->stream;
      cplx* V = ctx->ptr(off);
      cplx* x = V + (int64_t)m * n;
      cplx* y = x + n;
      cplx* z = y + n;
      launch_fill_zero(V, (int64_t)(m + 3) * n, s, &ctx->launches);
      std::vector<VecChunk> ch;
      for (int64_t st = 0; st < n; st += 8192) ch.push_back(VecChunk{st, (int)std::min<int64_t>(8192, n - st), 2.0f});
      const int B = 256;
      std::vector<CopyBlk> cb, cbt;
      for (int64_t st = 0; st + (int64_t)B * B <= n; st += (int64_t)B * B) {
        cb.push_back(CopyBlk{st, st, B, B, B, B, 0, 0, 1.25});
        cbt.push_back(CopyBlk{st, st, B, B, B, B, 1, 0, 1.25});
      }
      ctx->pool_aux.reserve(ch.size() * (sizeof(VecChunk) + 16) + 2 * cb.size() * sizeof(CopyBlk) + 8192, s);
      VecChunk* d_ch = upload(ctx->pool_aux, ch, s);
      CopyBlk* d_cb = upload(ctx->pool_aux, cb, s);
      CopyBlk* d_cbt = upload(ctx->pool_aux, cbt, s);
      double* d_part = (double*)ctx->pool_aux.take(ch.size() * 2 * sizeof(double));
      double* d_res = (double*)ctx->pool_aux.take(6 * sizeof(double));
      FH_CUDA(cudaMemsetAsync(d_res, 0, 6 * sizeof(double), s));
      unsigned* d_cnt = (unsigned*)ctx->pool_aux.take(sizeof(unsigned));
      FH_CUDA(cudaMemsetAsync(d_cnt, 0, sizeof(unsigned), s));
      FH_CUDA(cudaEventCreate(&e0));
      FH_CUDA(cudaEventCreate(&e1));
      std::vector<cplx> coef(m, make_double2(0.5, 0.25));
      const double nb = (double)cb.size() * B * B;
      const double bytes[7] = {32.0 * n, 48.0 * n, 32.0 * n, 16.0 * (m + 1) * n, 32.0 * nb, 32.0 * nb, 64.0 * n};
      for (int k = 0; k < 7; ++k) {
        for (int r = -2; r < reps; ++r) {
          if (r == 0) FH_CUDA(cudaEventRecord(e0, s));
          switch (k) {
            case 0: launch_wdot_fused(d_ch, (int)ch.size(), x, y, d_part, d_res, d_cnt, s, &ctx->launches); break;
            case 6:  // coefficients (d_res[2], d_res[3]) stay zero: the operands do not grow over the repetitions
              launch_lanczos_update(d_ch, (int)ch.size(), d_res + 2, d_res + 3, nullptr, 0.0, x, y, z, d_part, d_res + 4,
                                    d_cnt, s, &ctx->launches);
              break;
            case 1: launch_axpy(n, make_double2(0.5, 0.1), x, y, s, &ctx->launches); break;
            case 2: launch_scale(n, make_double2(0.5, 0.1), x, z, s, &ctx->launches); break;
            case 3: launch_lincomb(n, m, coef.data(), V, n, z, s, &ctx->launches); break;
            case 4: launch_copy_blocks(d_cb, (int)cb.size(), x, z, s, &ctx->launches); break;
            default: launch_copy_blocks(d_cbt, (int)cbt.size(), x, z, s, &ctx->launches); break;
          }
        }
        FH_CUDA(cudaEventRecord(e1, s));
        FH_CUDA(cudaEventSynchronize(e1));
        float ms = 0.f;
        FH_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        gbs[k] = bytes[k] * reps / (ms * 1e-3) * 1e-9;
      }
      FH_CUDA(cudaGetLastError());
    } catch (...) {
      if (e0) cudaEventDestroy(e0);
      if (e1) cudaEventDestroy(e1);
      ctx->alloc.release(off, (int64_t)(m + 3) * n);
      throw;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    ctx->alloc.release(off, (int64_t)(m + 3) * n);
  })
}

// ---- the Lanczos vector kernels and the scaled block copy on caller-supplied data (H6, H8): what expm_lanczos,
//      pack and unpack launch, with the chunk length the library would pick for a vector of n elements
static VecChunk* upload_chunks(fh_ctx* ctx, int64_t n, int nblk, const int64_t* blk_len, const int32_t* blk_weight,
                               int* nchunks, size_t extra_bytes) {
  std::vector<VecChunk> ch;
  const int cl = vec_chunk_len(n);
  int64_t pos = 0;
  for (int b = 0; b < nblk; ++b) {
    FH_REQUIRE(blk_len[b] >= 0 && blk_weight[b] >= 0, FH_EINVAL, "vector kernels: bad block table");
    for (int64_t s0 = 0; s0 < blk_len[b]; s0 += cl)
      ch.push_back(VecChunk{pos + s0, (int)std::min<int64_t>(cl, blk_len[b] - s0), (float)blk_weight[b]});
    pos += blk_len[b];
  }
  FH_REQUIRE(pos == n, FH_EINVAL, "vector kernels: block lengths do not add up to n");
  ctx->pool_aux.reserve(ch.size() * (sizeof(VecChunk) + 16) + extra_bytes + 8192, ctx->stream);
  *nchunks = (int)ch.size();
  return upload(ctx->pool_aux, ch, ctx->stream);
}

int fh_vec_wdot(fh_ctx* ctx, int64_t n, int nblk, const int64_t* blk_len, const int32_t* blk_weight, const void* x_dev,
                const void* y_dev, double* result) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && n > 0 && nblk > 0 && blk_len && blk_weight && x_dev && y_dev && result, FH_EINVAL, "fh_vec_wdot: bad argument");
    int nch = 0;
    VecChunk* d_ch = upload_chunks(ctx, n, nblk, blk_len, blk_weight, &nch, 0);
    double* d_part = (double*)ctx->pool_aux.take((size_t)nch * 2 * sizeof(double));
    double* d_res = (double*)ctx->pool_aux.take(2 * sizeof(double));
    unsigned* d_cnt = (unsigned*)ctx->pool_aux.take(sizeof(unsigned));
    FH_CUDA(cudaMemsetAsync(d_cnt, 0, sizeof(unsigned), ctx->stream));
    launch_wdot_fused(d_ch, nch, (const cplx*)x_dev, (const cplx*)y_dev, d_part, d_res, d_cnt, ctx->stream, &ctx->launches);
    ctx->ensure_pinned(2);
    FH_CUDA(cudaMemcpyAsync(ctx->h_pinned, d_res, 2 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    FH_CUDA(cudaStreamSynchronize(ctx->stream));
    result[0] = ctx->h_pinned[0];
    result[1] = ctx->h_pinned[1];
  })
}

int fh_vec_lanczos_update(fh_ctx* ctx, int64_t n, int nblk, const int64_t* blk_len, const int32_t* blk_weight, double a_raw,
                          double bj2, double bjm2, double tol, const void* uj_dev, const void* uprev_dev, void* w_dev,
                          double* norm2_out) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && n > 0 && nblk > 0 && blk_len && blk_weight && uj_dev && w_dev && norm2_out, FH_EINVAL,
               "fh_vec_lanczos_update: bad argument");
    int nch = 0;
    VecChunk* d_ch = upload_chunks(ctx, n, nblk, blk_len, blk_weight, &nch, 0);
    double* d_part = (double*)ctx->pool_aux.take((size_t)nch * 2 * sizeof(double));
    double* d_sc = (double*)ctx->pool_aux.take(8 * sizeof(double));
    unsigned* d_cnt = (unsigned*)ctx->pool_aux.take(sizeof(unsigned));
    FH_CUDA(cudaMemsetAsync(d_cnt, 0, sizeof(unsigned), ctx->stream));
    ctx->ensure_pinned(8);
    ctx->h_pinned[0] = a_raw;
    ctx->h_pinned[1] = bj2;
    ctx->h_pinned[2] = bjm2;
    FH_CUDA(cudaMemcpyAsync(d_sc, ctx->h_pinned, 3 * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    launch_lanczos_update(d_ch, nch, d_sc, bj2 > 0.0 ? d_sc + 1 : nullptr, (uprev_dev && bjm2 > 0.0) ? d_sc + 2 : nullptr, tol,
                          (const cplx*)uj_dev, (const cplx*)uprev_dev, (cplx*)w_dev, d_part, d_sc + 4, d_cnt, ctx->stream,
                          &ctx->launches);
    FH_CUDA(cudaMemcpyAsync(ctx->h_pinned + 4, d_sc + 4, 2 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    FH_CUDA(cudaStreamSynchronize(ctx->stream));
    *norm2_out = ctx->h_pinned[4];
  })
}

int fh_zgemm_split(fh_ctx* ctx, int M, int N, int nseg, const int32_t* K, const double* alpha, int conj_a, const void* A_dev,
                   const int64_t* a_off, const int32_t* a_sm, const int32_t* a_sk, const void* B_dev, const int64_t* b_off,
                   const int32_t* b_sk, const int32_t* b_sn, void* C_dev, int ldc) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && M > 0 && N > 0 && nseg >= 0 && ldc >= N && A_dev && B_dev && C_dev, FH_EINVAL, "fh_zgemm_split: bad argument");
    FH_REQUIRE(nseg == 0 || (K && alpha && a_off && a_sm && a_sk && b_off && b_sk && b_sn), FH_EINVAL,
               "fh_zgemm_split: segment arrays missing");
    Stage st;
    GemmOut o;
    o.c_off = 0;
    o.M = M;
    o.N = N;
    o.seg_begin = 0;
    o.seg_end = nseg;
    o.ldc = ldc;
    o.steps = 0;
    o.col0 = 0;
    for (int t = 0; t < nseg; ++t) {
      FH_REQUIRE(K[t] >= 0, FH_EINVAL, "fh_zgemm_split: negative K");
      GemmSeg g;
      g.a_off = a_off[t];
      g.b_off = b_off[t];
      g.K = K[t];
      g.a_sm = a_sm[t];
      g.a_sk = a_sk[t];
      g.b_sk = b_sk[t];
      g.b_sn = b_sn[t];
      g.pad = 0;
      g.alpha = alpha[t];
      st.segs.push_back(g);
    }
    st.mouts.push_back(o);
    std::vector<TcTile> tiles;
    std::vector<int> cb;
    build_tc_tiles(st, ctx->num_sms, tiles, cb);
    ctx->pool_aux.reserve(tiles.size() * sizeof(TcTile) + st.segs.size() * sizeof(GemmSeg) + cb.size() * 4 + 8192, ctx->stream);
    TcTile* d_t = upload(ctx->pool_aux, tiles, ctx->stream);
    int* d_cb = upload(ctx->pool_aux, cb, ctx->stream);
    GemmSeg* d_s = upload(ctx->pool_aux, st.segs, ctx->stream);
    launch_grouped_gemm_tc(d_t, d_cb, ctx->num_sms, (int)tiles.size(), d_s, conj_a ? 1 : 0, (const cplx*)A_dev, (const cplx*)B_dev,
                           (cplx*)C_dev, ctx->stream, &ctx->launches);
    FH_CUDA(cudaGetLastError());
    FH_CUDA(cudaStreamSynchronize(ctx->stream));  // tiles / segs are stack-owned
  })
}

int fh_vec_lincomb(fh_ctx* ctx, int64_t n, int m, const double* coef, const void* V_dev, int64_t stride, void* y_dev) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && n > 0 && m >= 1 && m <= 32 && coef && V_dev && y_dev && stride >= n, FH_EINVAL, "fh_vec_lincomb: bad argument");
    std::vector<cplx> c(m);
    for (int j = 0; j < m; ++j) c[j] = make_double2(coef[2 * j], coef[2 * j + 1]);
    launch_lincomb(n, m, c.data(), (const cplx*)V_dev, stride, (cplx*)y_dev, ctx->stream, &ctx->launches);
    FH_CUDA(cudaGetLastError());
  })
}

int fh_copy_blocks(fh_ctx* ctx, int nblk, const int64_t* src_off, const int64_t* dst_off, const int32_t* rows, const int32_t* cols,
                   const int32_t* ld_src, const int32_t* ld_dst, const int32_t* transpose, const double* scale,
                   const void* src_dev, void* dst_dev) {
  FH_TRY(ctx, {
    FH_REQUIRE(ctx && nblk > 0 && src_off && dst_off && rows && cols && ld_src && ld_dst && transpose && scale && src_dev &&
                   dst_dev && src_dev != dst_dev,
               FH_EINVAL, "fh_copy_blocks: bad argument");
    std::vector<CopyBlk> cb(nblk);
    for (int i = 0; i < nblk; ++i) {
      FH_REQUIRE(rows[i] >= 0 && cols[i] >= 0 && ld_src[i] >= cols[i] && ld_dst[i] >= (transpose[i] ? rows[i] : cols[i]), FH_EINVAL,
                 "fh_copy_blocks: bad block geometry");
      cb[i] = CopyBlk{src_off[i], dst_off[i], rows[i], cols[i], ld_src[i], ld_dst[i], transpose[i] ? 1 : 0, 0, scale[i]};
    }
    ctx->pool_aux.reserve(cb.size() * sizeof(CopyBlk) + 4096, ctx->stream);
    CopyBlk* d_cb = upload(ctx->pool_aux, cb, ctx->stream);
    launch_copy_blocks(d_cb, nblk, (const cplx*)src_dev, (cplx*)dst_dev, ctx->stream, &ctx->launches);
    FH_CUDA(cudaGetLastError());
  })
}

// host-only helpers for the CPU test-suite (symmetry layer without a GPU)
static fh::Stage g_host_st1, g_host_st2;

static const fh::SymMode* g_host_sym = &fh::SYM_SU2;
int fh_host_set_symmetry(int mode) {
  if (mode < 0 || mode > 1) return FH_EINVAL;
  g_host_sym = mode == 1 ? &fh::SYM_U1U1 : &fh::SYM_SU2;
  return FH_OK;
}

int fh_host_plan(int site, int nsite, double t_h, double U, int nl, const int32_t* bl, int nr, const int32_t* br,
                 int nLblk, const int32_t* Llab, int nRblk, const int32_t* Rlab) {
  try {
    fh::SymScope scope(g_host_sym);
    if ((nsite != 0 && nsite != 1 && nsite != 2) || !bl || !br || !Llab || !Rlab) return FH_EINVAL;
    Bond Bl, Br;
    for (int i = 0; i < nl; ++i) { Bl.sec.push_back(Sector{bl[3 * i], bl[3 * i + 1]}); Bl.d.push_back(bl[3 * i + 2]); }
    for (int i = 0; i < nr; ++i) { Br.sec.push_back(Sector{br[3 * i], br[3 * i + 1]}); Br.d.push_back(br[3 * i + 2]); }
    BlockTensor Le, Re, vec, Z;
    Le.nlab = Re.nlab = 5;
    for (int i = 0; i < nLblk; ++i) {
      const int32_t* l = Llab + 5 * i;
      Le.add(key_env(Sector{l[0], l[1]}, l[2], Sector{l[3], l[4]}), Bl.dim(Sector{l[0], l[1]}), Bl.dim(Sector{l[3], l[4]}));
    }
    for (int i = 0; i < nRblk; ++i) {
      const int32_t* l = Rlab + 5 * i;
      Re.add(key_env(Sector{l[0], l[1]}, l[2], Sector{l[3], l[4]}), Br.dim(Sector{l[0], l[1]}), Br.dim(Sector{l[3], l[4]}));
    }
    Le.finalize();
    Re.finalize();
    MpoSite W1, W2;
    mpo_site_table(site, t_h, U, W1);
    mpo_site_table(site + 1, t_h, U, W2);
    if (nsite == 0) {  // zero-site apply on the bond matrix C[c] (d_bl(c) x d_br(c)), NEXT-1
      vec.nlab = 2;
      for (size_t i = 0; i < Bl.sec.size(); ++i)
        if (Br.find(Bl.sec[i]) >= 0)
          vec.add(Key{Bl.sec[i].q, Bl.sec[i].tj, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, Bl.d[i], Br.dim(Bl.sec[i]));
      vec.finalize();
      emit_heff0(Le, Re, vec, Z, g_host_st1, g_host_st2);
    } else if (nsite == 2) {
      layout_theta(Bl, Br, vec);
      emit_heff2(Le, Re, vec, W1, W2, Z, g_host_st1, g_host_st2);
    } else {
      layout_site(Bl, Br, vec);
      emit_heff1(Le, Re, vec, W1, Z, g_host_st1, g_host_st2);
    }
    return FH_OK;
  } catch (...) {
    return FH_EINVAL;
  }
}

int fh_host_get_tasks(int stage, int* ntask, int* nout, int32_t* tuples, double* alpha, int64_t* flops) {
  if (stage != 1 && stage != 2) return FH_EINVAL;
  const Stage& st = stage == 1 ? g_host_st1 : g_host_st2;
  if (ntask) *ntask = (int)st.t_out.size();
  if (nout) *nout = (int)st.outs.size();
  if (flops) *flops = st.flops;
  for (size_t i = 0; i < st.t_out.size(); ++i) {
    if (tuples) { tuples[3 * i] = st.t_out[i]; tuples[3 * i + 1] = st.t_lhs[i]; tuples[3 * i + 2] = st.t_rhs[i]; }
    if (alpha) alpha[i] = st.t_alpha[i];
  }
  return FH_OK;
}

int fh_host_get_units(int stage, int* nunit, int32_t* units, int* nout, int32_t* outs, int64_t* dmma_padded) {
  if (stage != 1 && stage != 2) return FH_EINVAL;
  const Stage& st = stage == 1 ? g_host_st1 : g_host_st2;
  // the outputs the units tile: blocks merged with their compatible neighbours in a row panel (Stage::mouts)
  if (nunit) *nunit = (int)st.units.size();
  if (nout) *nout = (int)st.mouts.size();
  if (dmma_padded) *dmma_padded = st.dmma_padded;
  if (units) {
    // recover the output index of a unit from its c_off (merged outputs have distinct offsets)
    std::map<int64_t, int> by_off;
    for (size_t o = 0; o < st.mouts.size(); ++o) by_off[st.mouts[o].c_off] = (int)o;
    for (size_t i = 0; i < st.units.size(); ++i) {
      const GemmUnit& u = st.units[i];
      units[6 * i] = by_off.count(u.c_off) ? by_off[u.c_off] : -1;
      units[6 * i + 1] = u.m0;
      units[6 * i + 2] = u.n0;
      units[6 * i + 3] = u.shape >> 4;
      units[6 * i + 4] = u.shape & 15;
      units[6 * i + 5] = u.steps;
    }
  }
  if (outs)
    for (size_t o = 0; o < st.mouts.size(); ++o) {
      outs[3 * o] = st.mouts[o].M;
      outs[3 * o + 1] = st.mouts[o].N;
      outs[3 * o + 2] = st.mouts[o].steps;
    }
  return FH_OK;
}

int fh_host_get_tc_tiles(int stage, int grid, int static_side, int* ntile, int32_t* tiles, int32_t* cta_begin, int* nseg,
                         int* nimage_chunks, int64_t* seg_img, int64_t* seg_operand, int64_t* image_bytes) {
  if ((stage != 1 && stage != 2) || grid < 1) return FH_EINVAL;
  try {
    const Stage& st = stage == 1 ? g_host_st1 : g_host_st2;
    std::vector<TcTile> t;
    std::vector<int> cb;
    build_tc_tiles(st, grid, t, cb);
    if (ntile) *ntile = (int)t.size();
    if (nseg) *nseg = (int)st.segs.size();
    if (tiles) {
      std::map<int64_t, int> by_off;
      for (size_t o = 0; o < st.mouts.size(); ++o) by_off[st.mouts[o].c_off] = (int)o;
      for (size_t i = 0; i < t.size(); ++i) {
        tiles[6 * i] = by_off.count(t[i].c_off) ? by_off[t[i].c_off] : -1;
        tiles[6 * i + 1] = t[i].m0;
        tiles[6 * i + 2] = t[i].n0;
        tiles[6 * i + 3] = t[i].h;
        tiles[6 * i + 4] = t[i].w;
        tiles[6 * i + 5] = t[i].chunks;
      }
    }
    if (cta_begin)
      for (int b = 0; b <= grid; ++b) cta_begin[b] = cb[b];
    if (static_side == 1 || static_side == 2) {
      std::vector<int64_t> img;
      std::vector<TcPackChunk> pc;
      const int64_t bytes = build_tc_static(st, static_side == 1, img, pc);
      if (nimage_chunks) *nimage_chunks = (int)pc.size();
      if (image_bytes) *image_bytes = bytes;
      if (seg_img)
        for (size_t i = 0; i < img.size(); ++i) seg_img[i] = img[i];
      if (seg_operand)
        for (size_t i = 0; i < st.segs.size(); ++i) seg_operand[i] = static_side == 1 ? st.segs[i].a_off : st.segs[i].b_off;
    }
    return FH_OK;
  } catch (...) {
    return FH_EINVAL;
  }
}

double fh_canonical_weight(int tjc, int tjb) { return std::sqrt((double)(tjb + 1) / (double)(tjc + 1)); }

double fh_coef_left(int ta, int ts, int tc, int tk, int tr, int tkp, int tap, int tsp, int tcp) {
  return fh::coef_left(ta, ts, tc, tk, tr, tkp, tap, tsp, tcp);
}
double fh_coef_right(int tc, int ts, int tb, int tk, int tr, int tkp, int tcp, int tsp, int tbp) {
  return fh::coef_right(tc, ts, tb, tk, tr, tkp, tcp, tsp, tbp);
}

}  // extern "C"
