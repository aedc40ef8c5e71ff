// Internal declarations shared by the host layer and the kernels of libfh_b200.
// Product code: no dependency on oracle/ ("independence").
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>

#include <array>
#include <map>
#include <unordered_map>
#include <string>
#include <vector>

namespace fh {

typedef double2 cplx;  // complex128, interleaved (re, im)

// ----------------------------------------------------------------------------- labels
struct Sector {
  int q, tj;
  bool operator<(const Sector& o) const { return q != o.q ? q < o.q : tj < o.tj; }
  bool operator==(const Sector& o) const { return q == o.q && tj == o.tj; }
};

// Symmetry mode: the labels (q, tj) of the site multiplets and of the MPO bond multiplets.
//   SU2  (default): U(1)_spin x SU(2)_charge.  q = N_up - N_dn, tj = 2 T.  Site multiplets
//        s = 0 (+1,0) |up>, 1 (-1,0) |dn>, 2 (0,1/2) {|0>, eps |updn>}; MPO bond multiplets S, P, M, F (W = 4).
//   U1U1: U(1) x U(1), every multiplet one-dimensional (tj = 0, every
//        recoupling coefficient 1).  The two additive charges are packed into the one integer label,
//        q = (N_up - N_dn) + 64 (N - 1) per site (|N_up - N_dn| on a bond stays far below 32 for the chains in
//        reach, so the packing is unique).  Site states s = 0 |0>, 1 |up>, 2 |dn>, 3 |updn> = c+_up c+_dn |0>;
//        MPO bond states 0 = I, 1 = c+_up P, 2 = c+_dn P, 3 = c_up P, 4 = c_dn P, 5 = final (W = 6).
struct SymMode {
  int id;      // 0 SU2, 1 U1U1
  int ns, nw;  // site multiplets, MPO bond multiplets (the last one closes the MPO)
  int site_q[4], site_tj[4], mpo_q[6], mpo_tk[6];
};
const int MAX_NS = 4, MAX_NW = 6;
extern const SymMode SYM_SU2, SYM_U1U1;
// the mode of the calling thread: set for the duration of every API call from the context (SymScope)
const SymMode& sym();
struct SymScope {
  const SymMode* prev;
  explicit SymScope(const SymMode* m);
  ~SymScope();
};
#define SITE_Q (fh::sym().site_q)
#define SITE_TJ (fh::sym().site_tj)
#define MPO_Q (fh::sym().mpo_q)
#define MPO_TK (fh::sym().mpo_tk)

inline bool triangle(int t1, int t2, int t3) {
  int lo = t1 > t2 ? t1 - t2 : t2 - t1;
  return lo <= t3 && t3 <= t1 + t2 && ((t1 + t2 + t3) & 1) == 0;
}

// flattened label tuple, zero padded; compared lexicographically (== Python tuple order)
typedef std::array<int, 12> Key;
struct KeyHash {
  size_t operator()(const Key& k) const {
    uint64_t h = 1469598103934665603ull;
    for (int v : k) h = (h ^ (uint64_t)(uint32_t)v) * 1099511628211ull;
    return (size_t)(h ^ (h >> 29));
  }
};

struct Bond {
  std::vector<Sector> sec;  // sorted
  std::vector<int> d;
  int find(Sector s) const;
  int dim(Sector s) const {
    int i = find(s);
    return i < 0 ? 0 : d[i];
  }
  int chi_full() const;
  int chi_su2() const;
  int dmax() const;
};

struct BlockTensor {
  std::vector<Key> keys;  // sorted
  std::vector<int> rows, cols;
  std::vector<int64_t> off;  // element offsets relative to the tensor base
  // Leading dimension and first column of every block inside its row panel.  Blocks are dense row-major;
  // in the plain layout (finalize) each block is contiguous (ld = cols, col0 = 0).  The fused layouts of
  // the two-site vector and of its stage-1 intermediate (finalize_panels) put the blocks that share a
  // row-panel side by side in one matrix, so that a GEMM over several of them is ONE wider GEMM.
  std::vector<int> ld, col0;
  int64_t nelem = 0;
  int64_t base = -1;  // element offset in the arena, -1 = not allocated
  int nlab = 0;       // number of meaningful ints in each key
  std::unordered_map<Key, int, KeyHash> index;
  void clear();
  void add(const Key& k, int r, int c);  // append (caller adds in sorted order)
  void finalize();                       // plain layout: blocks contiguous, one after the other, in key order
  // fused layout: block i lies in panel `panel[i]` (panels numbered in memory order; all blocks of a panel
  // have the same row count) at column position `order[i]` within the panel (ranks need not be dense)
  void finalize_panels(const std::vector<int>& panel, const std::vector<int>& order);
  int find(const Key& k) const;
};

// reduced MPO of one site parity: val[w][w'][s'][s], rank2[w][w'] (-1 = absent)
struct MpoSite {
  double val[MAX_NW][MAX_NW][MAX_NS][MAX_NS];
  int rank2[MAX_NW][MAX_NW];
};

// recoupling coefficients, closed forms (su2.cpp)
double wigner6j(int ta, int tb, int tc, int td, int te, int tf);
double wigner9j(int a, int b, int c, int d, int e, int f, int g, int h, int i);
double coef_left(int ta, int ts, int tc, int tk, int tr, int tkp, int tap, int tsp, int tcp);
double coef_right(int tc, int ts, int tb, int tk, int tr, int tkp, int tcp, int tsp, int tbp);

// ----------------------------------------------------------------------------- GEMM task lists
enum OpA { OPA_N = 0, OPA_C = 1, OPA_H = 2 };  // as stored | conj | conj-transpose
enum OpB { OPB_N = 0, OPB_T = 1 };             // as stored | transpose

struct GemmOut {  // one output block C (M x N, row-major, leading dimension ldc)
  int64_t c_off;
  int M, N;
  int seg_begin, seg_end;
  int ldc, steps;  // steps = sum over segments of ceil(K / 4) (DMMA k-steps)
  int col0;        // first column inside its row panel (0 for a contiguous block)
};
struct GemmSeg {  // one K-segment: C += alpha * op(A) (M x K) * op(B) (K x N)
  int64_t a_off, b_off;   // element offsets of the operand blocks
  int K;
  int a_sm, a_sk;         // element strides of op(A): (m, k) -> a_off + m * a_sm + k * a_sk
  int b_sk, b_sn;         // element strides of op(B): (k, n) -> b_off + k * b_sk + n * b_sn
  int pad;
  double alpha;           // real recoupling coefficient x MPO scalar
};
// One warp's work: a (8*mt) x (8*nt) sub-tile of output block `out` over the whole K of that
// block (all its segments).  The output geometry is repeated here so that the kernel needs a
// single descriptor load per unit (96 bytes).  shape = mt * 16 + nt, mt * nt <= 16, mt, nt <= 8.
struct GemmUnit {
  int64_t c_off;
  int ldc, M, N, seg_begin, seg_end, steps, m0, n0, shape, pad;
  GemmSeg first;  // copy of segs[seg_begin]: the unit starts streaming after ONE descriptor load
};

// One tile of the warp-specialised kernel (zgemm_ws.cu): an (8 h) x (8 w) part (h, w <= 8) of output block
// `c_off`, worked on by a group of 2 x 2 consumer warps.  A tile covers the k range from k_begin inside segment
// seg_begin to k_end inside segment seg_end - 1 (both multiples of 16 or a segment end); a heavy tile is split
// along k into parts: kind 1 = a part that leaves its accumulators in scratch slot `slot`, kind 0 = the part
// that finally adds the `nparts` partial results of slots slot .. slot + nparts - 1 (in that order) and stores
// the block.  128 bytes; the first segment is repeated inside so that ONE load gives a producer everything it
// needs to start streaming.
struct WsTile {
  int64_t c_off;
  int ldc, M, N, m0, n0, h, w, seg_begin, seg_end, steps;
  GemmSeg first;
  int k_begin, k_end, kind, slot, nparts;
  // two stages in one launch (stage 2 reads what stage 1 writes): `stage` selects the operand set; a tile of
  // stage 1 that stores its block raises counter `sig` of its output panel when done; a tile of stage 2 may
  // start once the counters dep_id[dep_begin .. dep_begin + dep_count) have reached their targets
  int stage_sig;   // stage | (sig + 1) << 1
  int dep_begin, dep_count;
};
static_assert(sizeof(WsTile) == 128, "WsTile is one 128-byte line");

struct Stage {
  // host copies (canonical order) for heff_get_tasks and flops
  std::vector<int> t_out, t_lhs, t_rhs;
  std::vector<double> t_alpha;
  std::vector<double> t_scale;  // optional factor on alpha that is NOT part of the canonical list (vector gauge)
  std::vector<GemmOut> outs;    // one per output block, canonical order
  std::vector<GemmOut> mouts;   // outs with compatible neighbours in a row panel merged: what the units tile
  std::vector<GemmSeg> segs;
  std::vector<GemmUnit> units;  // sorted by work, heaviest first
  std::vector<WsTile> tiles;    // the same outputs cut into tiles for the warp-specialised kernel, heaviest first
  int n_slots = 0;              // scratch slots (WS_SLOT_ELEMS complex each) the k-split tiles of this stage need
  std::vector<int> out_mout;    // output block -> index into mouts (-1: empty block)
  std::vector<int> mout_tiles;  // per merged output: number of tiles that store (part of) it
  int opA = OPA_N, opB = OPB_N;
  int64_t flops = 0;
  int64_t dmma_padded = 0;  // DMMA.8x8x4 instructions the unit list issues (incl. ragged-edge padding)
  // device copies
  GemmSeg* d_segs = nullptr;
  GemmUnit* d_units = nullptr;
  WsTile* d_tiles = nullptr;
};

// weighted-vector chunk table (H6): contiguous chunk [start, start+len) carries weight w
struct VecChunk {
  int64_t start;
  int len;
  float w;  // 2j+1, small integer: exact in float
};

// Chunk length of the Lanczos vectors.  A chunk is one 256-thread CTA; a long chunk is a long chain of L2 round
// trips per thread (8192 elements = 32 loads), which is what a vector kernel on an L2-resident vector of a few
// MB waits for, so vectors up to 1 Mi elements get 1024-element chunks, up to 4 Mi 2048; HBM-sized vectors keep 8192 (fewer CTAs
// and partials).  One-site sweep at chi = 4096: 0.393 / 0.375 / 0.369 / 0.362 / 0.358 s with 8192 / 4096 / 2048 / 1024 / 512.
inline int vec_chunk_len(int64_t nelem) {
  return nelem > ((int64_t)4 << 20) ? 8192 : (nelem > ((int64_t)1 << 20) ? 2048 : 1024);
}

// pack / unpack copy descriptors (H8, H9)
struct CopyBlk {
  int64_t src_off, dst_off;
  int rows, cols, ld_src, ld_dst;
  int transpose_dst;  // write dst[c*ld_dst + r] instead of dst[r*ld_dst + c]
  int pad;
  double scale;
};

// ----------------------------------------------------------------------------- programmatic dependent launch
// The kernels of the Lanczos loop (grouped ZGEMM stage 1 / stage 2, weighted dot, three-term update, scale) follow
// one another on one stream, each depending on all of its predecessor.  They are launched with the
// programmatic-stream-serialisation attribute: every CTA issues griddepcontrol.launch_dependents at its start, so
// the next grid is set up and its CTAs move into warp slots the draining grid has freed, read their own
// descriptor (uploaded before either kernel started) and then block in griddepcontrol.wait, which returns only
// when the predecessor has completed and its writes are visible.  No kernel touches data a predecessor writes,
// or writes anything, before its wait.  FH_NO_PDL=1 in the environment launches them the plain way (A/B timing).
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// roles of a launch (bit mask; FH_PDL_MASK in the environment overrides which roles carry the attribute)
enum { PDL_GEMM_FIRST = 1, PDL_GEMM_SECOND = 2, PDL_WDOT = 4, PDL_UPDATE = 8, PDL_SCALE = 16, PDL_GEMM_OTHER = 32 };
const int PDL_DEFAULT_MASK = PDL_WDOT | PDL_UPDATE | PDL_SCALE;  // measured: see DESIGN.md 6.3
bool pdl_enabled(int role);
template <class... KArgs, class... Args>
inline void launch_pdl(int role, void (*kern)(KArgs...), int grid, int block, cudaStream_t s, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3((unsigned)block);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl_enabled(role) ? 1 : 0;
  cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}
#endif

// ----------------------------------------------------------------------------- kernel launchers (kernels.cu)
void launch_grouped_gemm(const Stage& st, const cplx* A, const cplx* B, cplx* C, cudaStream_t s,
                         int64_t* launch_counter, int pdl_role = 32 /* PDL_GEMM_OTHER */);
// warp-specialised persistent form (zgemm_ws.cu): d_counters = two zero-initialised unsigned (tile queue head,
// retired CTAs) that the kernel leaves at zero; grid = number of persistent CTAs (one per SM)
const int WS_SLOT_ELEMS = 4096;  // accumulators of one tile: 4 warps x 16 sub-tiles x 2 x 32 lanes
// scratch: n_slots * WS_SLOT_ELEMS elements; flags: n_slots counters, zero before the first launch, which the
// parts of launch number `epoch` (1, 2, ...) raise to 4 * epoch
void launch_grouped_gemm_ws(const Stage& st, const cplx* A, const cplx* B, cplx* C, unsigned* d_counters, int grid,
                            cplx* scratch, unsigned* flags, unsigned epoch, cudaStream_t s, int64_t* launch_counter);
// Two dependent stages (stage 2 reads C1 as its A or B operand) in ONE launch: tile queue = stage-1 tiles then
// stage-2 tiles; a stage-2 tile starts when the stage-1 panels it reads are complete (device counters).
struct WsPair {
  std::vector<WsTile> tiles;      // stage-1 tiles, then stage-2 tiles (segment indices into the joint array)
  std::vector<GemmSeg> segs;      // stage-1 segments, then stage-2 segments
  std::vector<int> dep_id;        // flattened dependency lists of the stage-2 tiles: stage-1 merged-output ids
  std::vector<unsigned> dep_target;  // arrivals per launch that complete that output (4 warps x its tiles)
  int n_dep_counters = 0;         // = number of stage-1 merged outputs
  int n_slots = 0;
  int conj1 = 0, conj2 = 0;
  WsTile* d_tiles = nullptr;
  GemmSeg* d_segs = nullptr;
  int* d_dep_id = nullptr;
  unsigned* d_dep_target = nullptr;
};
// which operand of stage 2 is stage 1's result: 0 = A (lhs), 1 = B (rhs)
void emit_ws_tiles(Stage& st);  // tile list of one stage (call before link_stages)
void link_stages(const Stage& st1, const Stage& st2, int mid_is_rhs2, WsPair& out);
void launch_grouped_gemm_ws_pair(const WsPair& pr, const cplx* A1, const cplx* B1, cplx* C1, const cplx* A2, const cplx* B2,
                                 cplx* C2, unsigned* d_counters, int grid, cplx* scratch, unsigned* flags,
                                 unsigned* dep_counters, unsigned epoch, cudaStream_t s, int64_t* launch_counter);
int ws_smem_bytes();
// warp-unit form with both stages in ONE launch (zgemm.cu): units of stage 1 then of stage 2, per unit its stage,
// the stage-1 output it signals (stage 1) or its dependency list (stage 2)
struct UnitLink {
  int stage, sig, dep_begin, dep_count;
};
struct UnitPair {
  std::vector<GemmUnit> units;
  std::vector<GemmSeg> segs;
  std::vector<UnitLink> link;
  std::vector<int> dep_id;
  std::vector<unsigned> dep_target;
  int n1 = 0, n_dep_counters = 0, conj1 = 0, conj2 = 0;
  GemmUnit* d_units = nullptr;
  GemmSeg* d_segs = nullptr;
  UnitLink* d_link = nullptr;
  int* d_dep_id = nullptr;
  unsigned* d_dep_target = nullptr;
};
void link_units(const Stage& st1, const Stage& st2, int mid_is_rhs2, UnitPair& out);
// dep_counters: n_dep_counters unsigned, zero before the first launch; launch number `epoch` (1, 2, ...) raises
// counter i to epoch * target_i
void launch_grouped_gemm_pair(const UnitPair& pr, const cplx* A1, const cplx* B1, cplx* C1, const cplx* A2, const cplx* B2,
                              cplx* C2, unsigned* dep_counters, unsigned epoch, cudaStream_t s, int64_t* launch_counter);
// split-precision form on tcgen05 (zgemm_tc.cu, NEXT-3): a tile = up to 128 x 128 of a merged output over all its
// segments (chunks = sum of ceil(K / 16)); same segment array, operands and results as the FP64 forms
struct TcTile {
  int64_t c_off;
  int ldc, m0, n0, h, w, seg_begin, seg_end, chunks, pad;
};
void build_tc_tiles(const Stage& st, int grid, std::vector<TcTile>& tiles, std::vector<int>& cta_begin);
// one 128-row x 16-k chunk of a static operand's panel images (zgemm_tc.cu): source element (row r, k) =
// X[src_off + r rs + k ks], `rows` x `kleft` of it valid, image of 32 KB at byte dst_off
struct TcPackChunk {
  int64_t src_off, dst_off;
  int rs, ks, rows, kleft;
};
int64_t build_tc_static(const Stage& st, bool a_side, std::vector<int64_t>& seg_img, std::vector<TcPackChunk>& chunks);
void launch_tc_pack(const TcPackChunk* d_chunks, int nchunks, const cplx* X, unsigned char* images, int conj, cudaStream_t s,
                    int64_t* launch_counter);
void launch_grouped_gemm_tc(const TcTile* d_tiles, const int* d_cta_begin, int grid, int ntiles, const GemmSeg* d_segs, int conjA,
                            const cplx* A, const cplx* B, cplx* C, cudaStream_t s, int64_t* launch_counter, int mode = 0,
                            const int64_t* d_seg_img = nullptr, const unsigned char* images = nullptr);
void launch_wdot(const VecChunk* d_chunks, int nchunks, const cplx* x, const cplx* y, double* d_partial,
                 double* d_result, cudaStream_t s, int64_t* launch_counter);
// y = y + a*x (a complex, from device scalar array coef[idx]*sign) etc.: see kernels.cu
void launch_axpy(int64_t n, cplx a, const cplx* x, cplx* y, cudaStream_t s, int64_t* lc);
void launch_scale(int64_t n, cplx a, const cplx* x, cplx* y, cudaStream_t s, int64_t* lc);  // y = a*x
// device-scalar Lanczos helpers: y -= d_coef[0] x;  y = x / sqrt(d_norm2[0]) (0 below tol), d_beta[0] = sqrt(d_norm2[0])
// one-launch forms for the Lanczos recurrence: d_counter is a zero-initialised unsigned that the kernels leave at zero
void launch_wdot_fused(const VecChunk* d_chunks, int nchunks, const cplx* x, const cplx* y, double* d_partial,
                       double* d_result, unsigned* d_counter, cudaStream_t s, int64_t* lc);
void launch_lanczos_update(const VecChunk* d_chunks, int nchunks, const double* d_a_raw, const double* d_bj2,
                           const double* d_bjm2, double tol, const cplx* vj, const cplx* vprev, cplx* w,
                           double* d_partial, double* d_result, unsigned* d_counter, cudaStream_t s, int64_t* lc);
void launch_scale_rsqrt_dev(int64_t n, const double* d_norm2, double tol, const cplx* x, cplx* y, double* d_beta,
                            cudaStream_t s, int64_t* lc);
void launch_lincomb(int64_t n, int m, const cplx* coef_host, const cplx* V, int64_t stride, cplx* y,
                    cudaStream_t s, int64_t* lc);  // y = sum_j coef[j] V[j]
void launch_copy_blocks(const CopyBlk* d_blks, int nblk, const cplx* src, cplx* dst, cudaStream_t s,
                        int64_t* lc);
// per-block weighted squared norms: out[i] = sum |x|^2 over block i
void launch_block_norms(const VecChunk* d_chunks, int nchunks, const cplx* x, double* d_out,
                        cudaStream_t s, int64_t* lc);
void launch_fill_zero(cplx* p, int64_t n, cudaStream_t s, int64_t* lc);
// calibration: register-only DMMA loop on 148*4 CTAs of 256 threads; returns the flops of one launch
double launch_dmma_peak(double* scratch, cudaStream_t s, int64_t* lc);

}  // namespace fh
