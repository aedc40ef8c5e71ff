// Split-precision form of the segmented grouped complex GEMM (
// reading A-18) on the fifth-generation tensor cores:
//     C_o (M x N) = sum_{t in seg(o)} alpha_t * op(A_t) (M x K_t) * op(B_t) (K_t x N),  alpha_t real,
// with complex128 operands and results in memory (the same task lists, layouts and launch interface as zgemm.cu)
// and the products taken as 3 x TF32:  x = hi + lo (+ 2^-22 |x|; hi, lo = x and x - hi rounded to 11 significant
// bits),  a b ~ hi hi + hi lo + lo hi, accumulated in float32 in tensor memory (oracle/splitprec.py states the
// arithmetic and its two error bounds).
//
// One persistent CTA per SM, 22 warps, four roles that meet only at mbarriers:
//   * The operand of a stage that does not change between applies (an environment: op(A) of stage 1, op(B) of
//     stage 2) is converted ONCE per plan by tc_pack_kernel into PANEL IMAGES -- per 128-row tile and 16-k chunk
//     the four TF32 planes (re hi, re lo, im hi, im lo) in exactly the shared-memory layout below, 32 KB, zero
//     padded, one image per distinct block however many segments read it -- and ONE thread streams them into the
//     ring with cp.async.bulk onto the stage's mbarrier (complete_tx).
//   * 16 CONVERTER warps (one thread = one row of the 128-row panel and 4 of a chunk's 16 k) load the operand that
//     changes with every apply as complex128 straight from its blocks (any stride pair, zero beyond a segment's K;
//     the loads of the next chunk of the segment are in flight while the current one is converted), fold the
//     segment's alpha (and the conjugation sign) into it, split every real number into its two TF32 parts, and
//     write the four planes of the panel to shared memory in the K-major no-swizzle core-matrix layout
//     tcgen05.mma reads (8 rows x 16 B per core matrix; 128 B between row groups, 2048 B between k quads).
//     Without a static operand (fh_zgemm_split) 8 + 8 converter warps take the A and the B panel, alpha on A.
//   * ONE thread issues the MMAs: per 8 k, 12 x tcgen05.mma.kind::tf32 (M = 128, N = the tile width rounded up
//     to 16): Re C += Ar Br - Ai Bi, Im C += Ar Bi + Ai Br, each as hi hi + hi lo + lo hi; the minus sign is the
//     negate-A bit of the instruction descriptor.  Accumulators: 2 x 128 float32 columns of tensor memory per
//     tile, double buffered (all 512 columns).  tcgen05.commit hands a shared-memory stage (3 x 64 KB) back to the
//     producers and, after the last chunk of a tile, the accumulator buffer over to the epilogue.
//   * 4 EPILOGUE warps (warp w owns TMEM lanes 32 w ... 32 w + 31 = tile rows) read the accumulators with
//     tcgen05.ld (32 lanes x 32 columns per instruction), widen them to double and store complex128.
// All K segments of an output accumulate in tensor memory (alpha is inside the converted operand), so there is one
// epilogue per tile.  Tiles are dealt to the CTAs on the host (heaviest first to the least loaded); a tile without
// segments is stored as zeros.  Deterministic: fixed tile -> CTA map, fixed k order, one accumulator per output
// element.  Measurements, ablations and what was tried and dropped: DESIGN.md 6.8, profiles/r2_zgemm_tc_ncu.md.
#include "fh_internal.hpp"

#include <algorithm>
#include <map>
#include <tuple>

namespace fh {

namespace {

constexpr int TC_STAGES = 3;
constexpr int TC_KC = 16;                          // k per chunk = two MMA k-steps of 8
constexpr int TC_PLANE = 128 * TC_KC * 4;          // one TF32 plane of a panel: 128 rows x 16 k
constexpr int TC_OPERAND = 4 * TC_PLANE;           // re hi, re lo, im hi, im lo
constexpr int TC_STAGE_BYTES = 2 * TC_OPERAND;     // A panel + B panel = 64 KB
constexpr int TC_EPI_WARPS = 4, TC_CONV_WARPS = 16;
constexpr int TC_MMA_WARP = TC_EPI_WARPS;          // warp 4
constexpr int TC_THREADS = 32 * (TC_EPI_WARPS + 1 + TC_CONV_WARPS + 1);  // + the warp whose lane 0 issues the bulk copies
constexpr int TC_NBAR = 2 * TC_STAGES + 4;
constexpr int TC_SMEM_BYTES = TC_STAGES * TC_STAGE_BYTES + 8 * TC_NBAR + 16;
constexpr uint32_t TC_LBO = 2048, TC_SBO = 128;    // byte strides between core matrices along k / along rows

__device__ __forceinline__ void mbar_init(uint32_t a, int count) {
  asm volatile("mbarrier.init.shared.b64 [%0], %1;" ::"r"(a), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t a) {
  asm volatile("mbarrier.arrive.shared.b64 _, [%0];" ::"r"(a) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t a, uint32_t parity) {
  uint32_t ok = 0;
  while (!ok) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(a), "r"(parity)
        : "memory");
  }
}
// x -> (hi, lo), both TF32 numbers in float32 bit patterns, with integer arithmetic on the bits of the double
// (F2F.F32.F64 runs at 8 per clock and SM on this part, measured; the integer pipe at 64+):
//   round11(v): v rounded to 11 significant bits, ties away from zero = add half a unit (bit 41 of the double =
//               bit 9 of its high word) and clear the 42 bits below; the low word plays no part;
//   hi = round11(x), lo = round11(x - hi) (the difference is exact in double).
// A double with <= 11 significant bits becomes a float32 by re-biasing the exponent (1023 -> 127) and moving the
// 20 mantissa bits of the high word up by 3; magnitudes below 2^-126 become (sub)zero bits: max(., 0).
__device__ __forceinline__ uint32_t round11_hiword(double v) { return ((uint32_t)__double2hiint(v) + 0x200u) & 0xFFFFFC00u; }
__device__ __forceinline__ uint32_t f32_bits_of_hiword(uint32_t hw) {
  const int e = max((int)(hw & 0x7FFFFFFFu) - 0x38000000, 0);
  return ((uint32_t)e << 3) | (hw & 0x80000000u);
}
__device__ __forceinline__ void split_tf32(double x, uint32_t& hi, uint32_t& lo) {
  const uint32_t hh = round11_hiword(x);
  hi = f32_bits_of_hiword(hh);
  lo = f32_bits_of_hiword(round11_hiword(x - __hiloint2double((int)hh, 0)));
}
__device__ __forceinline__ void sts128(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
// shared-memory matrix descriptor: K-major, no swizzle, version 1 (sm_100)
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr) {
  return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)(TC_LBO >> 4) << 16) | ((uint64_t)(TC_SBO >> 4) << 32) |
         ((uint64_t)1 << 46);
}
// instruction descriptor: D float32, A / B TF32, both K-major, M = 128, N = n
__device__ __forceinline__ uint32_t instr_desc(int n, int neg_a) {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)neg_a << 13) | ((uint32_t)(n >> 3) << 17) | (8u << 24);
}
__device__ __forceinline__ void mma_tf32(uint32_t d_tmem, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void mma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
        "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
        "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
        "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr)
      : "memory");
}

struct TcSmem {
  uint32_t data, full, empty, tfull, tempty, tptr;
  __device__ __forceinline__ uint32_t a_panel(int s) const { return data + s * TC_STAGE_BYTES; }
  __device__ __forceinline__ uint32_t b_panel(int s) const { return data + s * TC_STAGE_BYTES + TC_OPERAND; }
};

// ------------------------------------------------------------------------------------------------ converters
// One thread = one row of its panel and NK of the chunk's 16 k: NK complex128 -> 4 planes x NK TF32.
// op(A)(m, k) = A[a_off + m a_sm + k a_sk], op(B)(k, n) = B[b_off + k b_sk + n b_sn]: both panels are "row x k".
// `dst` = address of (row, first k of this thread) in plane 0; generic address space: shared memory in the GEMM
// kernel, global memory in the kernel that packs a static operand once per plan (same image either way).
template <int NK>
__device__ __forceinline__ void load_row(const cplx* __restrict__ p, int64_t k_stride, int k_left, cplx (&z)[NK]) {
#pragma unroll
  for (int i = 0; i < NK; ++i) {
    z[i] = make_double2(0.0, 0.0);
    if (i < k_left) z[i] = __ldg(p + (int64_t)i * k_stride);
  }
}
template <int NK, bool SCALE, bool TO_SHARED>
__device__ __forceinline__ void convert_store(const cplx (&z)[NK], double scale, double im_scale, uint32_t dst_s, unsigned char* dst_g) {
#pragma unroll
  for (int q = 0; q < NK / 4; ++q) {
    uint32_t rh[4], rl[4], ih[4], il[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      split_tf32(SCALE ? z[4 * q + i].x * scale : z[4 * q + i].x, rh[i], rl[i]);
      split_tf32(SCALE ? z[4 * q + i].y * im_scale : z[4 * q + i].y, ih[i], il[i]);
    }
    if (TO_SHARED) {
      const uint32_t a = dst_s + q * TC_LBO;
      sts128(a, rh[0], rh[1], rh[2], rh[3]);
      sts128(a + TC_PLANE, rl[0], rl[1], rl[2], rl[3]);
      sts128(a + 2 * TC_PLANE, ih[0], ih[1], ih[2], ih[3]);
      sts128(a + 3 * TC_PLANE, il[0], il[1], il[2], il[3]);
    } else {
      unsigned char* a = dst_g + q * TC_LBO;
      *reinterpret_cast<uint4*>(a) = make_uint4(rh[0], rh[1], rh[2], rh[3]);
      *reinterpret_cast<uint4*>(a + TC_PLANE) = make_uint4(rl[0], rl[1], rl[2], rl[3]);
      *reinterpret_cast<uint4*>(a + 2 * TC_PLANE) = make_uint4(ih[0], ih[1], ih[2], ih[3]);
      *reinterpret_cast<uint4*>(a + 3 * TC_PLANE) = make_uint4(il[0], il[1], il[2], il[3]);
    }
  }
}

// MODE 0: both operands converted in the loop (8 + 8 warps, 8 k per thread), alpha folded into A.
// MODE 1: A is STATIC (an environment: converted once per plan into panel images, streamed by cp.async.bulk), all
//         16 converter warps work on B (4 k per thread) and fold alpha into it.
// MODE 2: B is static, all 16 converter warps work on A and fold alpha (and the conjugation sign) into it.
template <int NK, bool SCALE, bool TO_SHARED>
__device__ __forceinline__ void convert_row(const cplx* __restrict__ p, int64_t k_stride, int k_left, double scale, double im_scale,
                                            uint32_t dst_s, unsigned char* dst_g) {
  cplx z[NK];
  load_row<NK>(p, k_stride, k_left, z);
  convert_store<NK, SCALE, TO_SHARED>(z, scale, im_scale, dst_s, dst_g);
}

template <int MODE>
__device__ __forceinline__ void converter_loop(const TcTile* __restrict__ tiles, const int* __restrict__ cta_begin, const GemmSeg* __restrict__ segs,
                                               const cplx* __restrict__ A, const cplx* __restrict__ B, double conj_sign,
                                               const TcSmem& sm, int ct) {
  const bool is_a = MODE == 0 ? ct < 256 : MODE == 2;
  const int row = ct & 127;
  const int kpart = MODE == 0 ? 8 * ((ct >> 7) & 1) : 4 * (ct >> 7);  // first k of this thread inside a chunk
  uint32_t g = 0;  // chunks produced so far by this CTA
  for (int t = cta_begin[blockIdx.x], t_end = cta_begin[blockIdx.x + 1]; t < t_end; ++t) {
    const TcTile tl = tiles[t];
    const bool row_valid = is_a ? row < tl.h : row < tl.w;
    for (int si = tl.seg_begin; si < tl.seg_end; ++si) {
      const GemmSeg sg = segs[si];
      const cplx* base = is_a ? A + sg.a_off + (int64_t)(tl.m0 + row) * sg.a_sm : B + sg.b_off + (int64_t)(tl.n0 + row) * sg.b_sn;
      const int64_t ks = is_a ? sg.a_sk : sg.b_sk;
      const bool scaled = MODE == 0 ? is_a : true;
      const double scale = scaled ? sg.alpha : 1.0, im_scale = scaled ? sg.alpha * (is_a ? conj_sign : 1.0) : 1.0;
      // MODE 1 / 2: the loads of the next chunk of the segment are issued before this chunk is converted (and before the
      // wait for its stage), so a thread's load latency overlaps its own conversion work
      cplx zc[4], zn[4];
      if (MODE != 0 && row_valid) load_row<4>(base + (int64_t)kpart * ks, ks, sg.K - kpart, zc);
      for (int k0 = 0; k0 < sg.K; k0 += TC_KC, ++g) {
        const int s = g % TC_STAGES;
        if (MODE != 0 && row_valid && k0 + TC_KC < sg.K)
          load_row<4>(base + (int64_t)(k0 + TC_KC + kpart) * ks, ks, sg.K - k0 - TC_KC - kpart, zn);
        mbar_wait(sm.empty + 8 * s, ((g / TC_STAGES) & 1) ^ 1);
        if (row_valid) {  // rows beyond the tile edge only feed accumulator rows / columns that are never stored
          const uint32_t dst = (is_a ? sm.a_panel(s) : sm.b_panel(s)) + (uint32_t)(row * 16) + (uint32_t)(kpart >> 2) * TC_LBO;
          if (MODE == 0) {
            const cplx* p = base + (int64_t)(k0 + kpart) * ks;
            if (is_a) convert_row<8, true, true>(p, ks, sg.K - k0 - kpart, scale, im_scale, dst, nullptr);
            else convert_row<8, false, true>(p, ks, sg.K - k0 - kpart, 1.0, 1.0, dst, nullptr);
          } else {
            convert_store<4, true, true>(zc, scale, im_scale, dst, nullptr);
#pragma unroll
            for (int i = 0; i < 4; ++i) zc[i] = zn[i];
          }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy stores -> visible to the MMA (async proxy)
        mbar_arrive(sm.full + 8 * s);
      }
    }
  }
}

// MODE 1 / 2: one thread streams the static operand's panel images (32 KB per chunk, laid out exactly as the
// shared-memory panel) with cp.async.bulk; the copy completes on the stage's full barrier (complete_tx).
template <int MODE>
__device__ __forceinline__ void bulk_loop(const TcTile* __restrict__ tiles, const int* __restrict__ cta_begin, const GemmSeg* __restrict__ segs,
                                          const int64_t* __restrict__ seg_img, const unsigned char* __restrict__ images,
                                          const TcSmem& sm) {
  uint32_t g = 0;
  for (int t = cta_begin[blockIdx.x], t_end = cta_begin[blockIdx.x + 1]; t < t_end; ++t) {
    const TcTile tl = tiles[t];
    const int rt = (MODE == 1 ? tl.m0 : tl.n0) >> 7;  // row tile of the static operand this output tile reads
    for (int si = tl.seg_begin; si < tl.seg_end; ++si) {
      const int K = segs[si].K;
      const int nch = (K + TC_KC - 1) / TC_KC;
      const unsigned char* src = images + seg_img[si] + (int64_t)rt * nch * TC_OPERAND;
      for (int c = 0; c < nch; ++c, ++g, src += TC_OPERAND) {
        const int s = g % TC_STAGES;
        mbar_wait(sm.empty + 8 * s, ((g / TC_STAGES) & 1) ^ 1);
        const uint32_t bar = sm.full + 8 * s, dst = MODE == 1 ? sm.a_panel(s) : sm.b_panel(s);
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(TC_OPERAND) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(dst), "l"(src), "r"(TC_OPERAND), "r"(bar)
                     : "memory");
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------ MMA issuer
__device__ __forceinline__ void mma_loop(const TcTile* __restrict__ tiles, const int* __restrict__ cta_begin, const TcSmem& sm, uint32_t tmem) {
  uint32_t g = 0, tt = 0;
  for (int t = cta_begin[blockIdx.x], t_end = cta_begin[blockIdx.x + 1]; t < t_end; ++t) {
    const TcTile tl = tiles[t];
    if (tl.chunks == 0) continue;
    const int n_inst = max(16, (tl.w + 15) & ~15);
    const uint32_t id_pos = instr_desc(n_inst, 0), id_neg = instr_desc(n_inst, 1);
    const uint32_t buf = tt & 1;
    mbar_wait(sm.tempty + 8 * buf, ((tt >> 1) & 1) ^ 1);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t d_re = tmem + buf * 256, d_im = d_re + 128;
    for (int c = 0; c < tl.chunks; ++c, ++g) {
      const int s = g % TC_STAGES;
      mbar_wait(sm.full + 8 * s, (g / TC_STAGES) & 1);
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
      for (int j = 0; j < TC_KC / 8; ++j) {
        const uint32_t pa = sm.a_panel(s) + j * 2 * TC_LBO, pb = sm.b_panel(s) + j * 2 * TC_LBO;
        const uint64_t ar_h = smem_desc(pa), ar_l = smem_desc(pa + TC_PLANE), ai_h = smem_desc(pa + 2 * TC_PLANE),
                       ai_l = smem_desc(pa + 3 * TC_PLANE);
        const uint64_t br_h = smem_desc(pb), br_l = smem_desc(pb + TC_PLANE), bi_h = smem_desc(pb + 2 * TC_PLANE),
                       bi_l = smem_desc(pb + 3 * TC_PLANE);
        const uint32_t acc = (c | j) != 0;
        // Re C += Ar Br - Ai Bi
        mma_tf32(d_re, ar_h, br_h, id_pos, acc);
        mma_tf32(d_re, ar_h, br_l, id_pos, 1);
        mma_tf32(d_re, ar_l, br_h, id_pos, 1);
        mma_tf32(d_re, ai_h, bi_h, id_neg, 1);
        mma_tf32(d_re, ai_h, bi_l, id_neg, 1);
        mma_tf32(d_re, ai_l, bi_h, id_neg, 1);
        // Im C += Ar Bi + Ai Br
        mma_tf32(d_im, ar_h, bi_h, id_pos, acc);
        mma_tf32(d_im, ar_h, bi_l, id_pos, 1);
        mma_tf32(d_im, ar_l, bi_h, id_pos, 1);
        mma_tf32(d_im, ai_h, br_h, id_pos, 1);
        mma_tf32(d_im, ai_h, br_l, id_pos, 1);
        mma_tf32(d_im, ai_l, br_h, id_pos, 1);
      }
      mma_commit(sm.empty + 8 * s);  // the stage is free once these MMAs have read it
    }
    mma_commit(sm.tfull + 8 * buf);  // accumulators of the tile complete
    ++tt;
  }
}

// ------------------------------------------------------------------------------------------------ epilogue
__device__ __forceinline__ void epilogue_loop(const TcTile* __restrict__ tiles, const int* __restrict__ cta_begin, cplx* __restrict__ C,
                                              const TcSmem& sm, uint32_t tmem, int warp, int lane) {
  const int row = 32 * warp + lane;
  uint32_t tt = 0;
  for (int t = cta_begin[blockIdx.x], t_end = cta_begin[blockIdx.x + 1]; t < t_end; ++t) {
    const TcTile tl = tiles[t];
    cplx* crow = C + tl.c_off + (int64_t)(tl.m0 + row) * tl.ldc + tl.n0;
    if (tl.chunks == 0) {  // an output without contributions
      if (row < tl.h)
        for (int c = 0; c < tl.w; ++c) crow[c] = make_double2(0.0, 0.0);
      continue;
    }
    const uint32_t buf = tt & 1;
    mbar_wait(sm.tfull + 8 * buf, (tt >> 1) & 1);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t t_re = tmem + ((uint32_t)(32 * warp) << 16) + buf * 256;
    for (int c0 = 0; c0 < tl.w; c0 += 32) {
      uint32_t re[32], im[32];
      tmem_ld32(t_re + c0, re);
      tmem_ld32(t_re + 128 + c0, im);
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
      if (row < tl.h) {
#pragma unroll
        for (int i = 0; i < 32; ++i)
          if (c0 + i < tl.w) crow[c0 + i] = make_double2((double)__uint_as_float(re[i]), (double)__uint_as_float(im[i]));
      }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    mbar_arrive(sm.tempty + 8 * buf);
    ++tt;
  }
}

template <int MODE>
__global__ void __launch_bounds__(TC_THREADS, 1)
    grouped_zgemm_tc_kernel(const TcTile* __restrict__ tiles, const int* __restrict__ cta_begin, const GemmSeg* __restrict__ segs,
                            const cplx* __restrict__ A, const cplx* __restrict__ B, cplx* __restrict__ C, int conjA,
                            const int64_t* __restrict__ seg_img, const unsigned char* __restrict__ images) {
  extern __shared__ __align__(1024) unsigned char tc_smem[];
  TcSmem sm;
  sm.data = (uint32_t)__cvta_generic_to_shared(tc_smem);
  sm.full = sm.data + TC_STAGES * TC_STAGE_BYTES;
  sm.empty = sm.full + 8 * TC_STAGES;
  sm.tfull = sm.empty + 8 * TC_STAGES;
  sm.tempty = sm.tfull + 16;
  sm.tptr = sm.tempty + 16;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < TC_STAGES; ++s) {
      // every converter thread arrives after its own stores; with a static operand also the thread that starts
      // the bulk copy (arrive.expect_tx; the bytes complete the phase)
      mbar_init(sm.full + 8 * s, 32 * TC_CONV_WARPS + (MODE != 0 ? 1 : 0));
      mbar_init(sm.empty + 8 * s, 1);                  // tcgen05.commit
    }
    for (int b = 0; b < 2; ++b) {
      mbar_init(sm.tfull + 8 * b, 1);                  // tcgen05.commit
      mbar_init(sm.tempty + 8 * b, 32 * TC_EPI_WARPS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == TC_MMA_WARP) {  // all 512 columns: two accumulator buffers of 2 x 128 (one CTA per SM, nobody to share with)
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sm.tptr), "r"(512) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  uint32_t tmem;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem) : "r"(sm.tptr) : "memory");

  if (warp < TC_EPI_WARPS) {
    epilogue_loop(tiles, cta_begin, C, sm, tmem, warp, lane);
  } else if (warp == TC_MMA_WARP) {
    if (lane == 0) mma_loop(tiles, cta_begin, sm, tmem);
    __syncwarp();
  } else if (warp <= TC_MMA_WARP + TC_CONV_WARPS) {
    converter_loop<MODE>(tiles, cta_begin, segs, A, B, conjA ? -1.0 : 1.0, sm, (int)threadIdx.x - 32 * (TC_MMA_WARP + 1));
  } else {
    if (MODE != 0 && lane == 0) bulk_loop<MODE>(tiles, cta_begin, segs, seg_img, images, sm);
    __syncwarp();
  }

  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == TC_MMA_WARP)
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512) : "memory");
}

// Packs a static operand once per plan: one CTA per panel image chunk (128 rows x 16 k, 4 planes, 32 KB, zero padded),
// one thread per row; no alpha (the converters of the other operand carry it), conjugation as the stage says.
__global__ void __launch_bounds__(128) tc_pack_kernel(const TcPackChunk* __restrict__ chunks, const cplx* __restrict__ X,
                                                      unsigned char* __restrict__ images, double im_sign) {
  const TcPackChunk c = chunks[blockIdx.x];
  const int row = threadIdx.x;
  unsigned char* dst = images + c.dst_off + row * 16;
  const cplx* p = X + c.src_off + (int64_t)row * c.rs;
  convert_row<16, true, false>(p, c.ks, row < c.rows ? c.kleft : 0, 1.0, im_sign, 0u, dst);
}

}  // namespace

// 128 x 128 tiles of the merged outputs, dealt to `grid` persistent CTAs heaviest first to the least loaded CTA
// (weight = chunks x a mix of the converter cost, which does not depend on the width, and the MMA cost, which
// does); the tiles of CTA b are tiles[cta_begin[b] .. cta_begin[b + 1]), heaviest first
void build_tc_tiles(const Stage& st, int grid, std::vector<TcTile>& tiles, std::vector<int>& cta_begin) {
  std::vector<TcTile> all;
  for (const GemmOut& o : st.mouts) {
    int chunks = 0;
    for (int s = o.seg_begin; s < o.seg_end; ++s) chunks += (st.segs[s].K + TC_KC - 1) / TC_KC;
    for (int m0 = 0; m0 < o.M; m0 += 128)
      for (int n0 = 0; n0 < o.N; n0 += 128) {
        TcTile t;
        t.c_off = o.c_off;
        t.ldc = o.ldc;
        t.m0 = m0;
        t.n0 = n0;
        t.h = std::min(128, o.M - m0);
        t.w = std::min(128, o.N - n0);
        t.seg_begin = o.seg_begin;
        t.seg_end = o.seg_end;
        t.chunks = chunks;
        t.pad = 0;
        all.push_back(t);
      }
  }
  auto weight = [](const TcTile& t) { return (int64_t)t.chunks * (128 + ((t.w + 15) & ~15)) + 64; };
  std::stable_sort(all.begin(), all.end(), [&](const TcTile& a, const TcTile& b) { return weight(a) > weight(b); });
  grid = std::max(1, grid);
  std::vector<std::vector<int>> mine(grid);
  std::vector<std::pair<int64_t, int>> heap;  // (-load, cta): max-heap on -load = least loaded first
  for (int b = 0; b < grid; ++b) heap.push_back({0, -b});
  std::make_heap(heap.begin(), heap.end());
  for (size_t i = 0; i < all.size(); ++i) {
    std::pop_heap(heap.begin(), heap.end());
    auto& top = heap.back();
    mine[-top.second].push_back((int)i);
    top.first -= weight(all[i]);
    std::push_heap(heap.begin(), heap.end());
  }
  tiles.clear();
  cta_begin.assign(grid + 1, 0);
  for (int b = 0; b < grid; ++b) {
    for (int i : mine[b]) tiles.push_back(all[i]);
    cta_begin[b + 1] = (int)tiles.size();
  }
}

// Panel images of the static operand of a stage (a_side: op(A), else op(B)): one image per distinct operand region
// (offset, strides, K, rows) -- segments that read the same environment block share it -- cut into row tiles of 128
// and chunks of 16 k.  seg_img[s] = byte offset of the image of segment s; chunks = what tc_pack_kernel converts.
int64_t build_tc_static(const Stage& st, bool a_side, std::vector<int64_t>& seg_img, std::vector<TcPackChunk>& chunks) {
  struct Key {
    int64_t off;
    int rs, ks, K, rows;
    bool operator<(const Key& o) const { return std::tie(off, rs, ks, K, rows) < std::tie(o.off, o.rs, o.ks, o.K, o.rows); }
  };
  std::map<Key, int64_t> seen;
  seg_img.assign(st.segs.size(), -1);  // segments of outputs that were merged into a neighbour are not read by any tile
  chunks.clear();
  int64_t bytes = 0;
  for (const GemmOut& o : st.mouts)
    for (int s = o.seg_begin; s < o.seg_end; ++s) {
      const GemmSeg& g = st.segs[s];
      const Key k{a_side ? g.a_off : g.b_off, a_side ? g.a_sm : g.b_sn, a_side ? g.a_sk : g.b_sk, g.K, a_side ? o.M : o.N};
      auto it = seen.find(k);
      if (it == seen.end()) {
        it = seen.emplace(k, bytes).first;
        const int nrt = (k.rows + 127) / 128, nch = (k.K + TC_KC - 1) / TC_KC;
        for (int rt = 0; rt < nrt; ++rt)
          for (int c = 0; c < nch; ++c) {
            TcPackChunk pc;
            pc.src_off = k.off + (int64_t)rt * 128 * k.rs + (int64_t)c * TC_KC * k.ks;
            pc.dst_off = bytes;
            pc.rs = k.rs;
            pc.ks = k.ks;
            pc.rows = std::min(128, k.rows - rt * 128);
            pc.kleft = std::min(TC_KC, k.K - c * TC_KC);
            chunks.push_back(pc);
            bytes += TC_OPERAND;
          }
      }
      seg_img[s] = it->second;
    }
  return bytes;
}

void launch_tc_pack(const TcPackChunk* d_chunks, int nchunks, const cplx* X, unsigned char* images, int conj, cudaStream_t s,
                    int64_t* lc) {
  if (nchunks == 0) return;
  tc_pack_kernel<<<nchunks, 128, 0, s>>>(d_chunks, X, images, conj ? -1.0 : 1.0);
  ++*lc;
}

// mode 0: both operands converted in the loop; 1: op(A) from panel images; 2: op(B) from panel images
void launch_grouped_gemm_tc(const TcTile* d_tiles, const int* d_cta_begin, int grid, int ntiles, const GemmSeg* d_segs, int conjA,
                            const cplx* A, const cplx* B, cplx* C, cudaStream_t s, int64_t* lc, int mode, const int64_t* d_seg_img,
                            const unsigned char* images) {
  if (ntiles == 0) return;
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(grouped_zgemm_tc_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, TC_SMEM_BYTES);
    cudaFuncSetAttribute(grouped_zgemm_tc_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, TC_SMEM_BYTES);
    cudaFuncSetAttribute(grouped_zgemm_tc_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, TC_SMEM_BYTES);
    attr_set = true;
  }
  if (mode == 1)
    grouped_zgemm_tc_kernel<1><<<grid, TC_THREADS, TC_SMEM_BYTES, s>>>(d_tiles, d_cta_begin, d_segs, A, B, C, conjA, d_seg_img, images);
  else if (mode == 2)
    grouped_zgemm_tc_kernel<2><<<grid, TC_THREADS, TC_SMEM_BYTES, s>>>(d_tiles, d_cta_begin, d_segs, A, B, C, conjA, d_seg_img, images);
  else
    grouped_zgemm_tc_kernel<0><<<grid, TC_THREADS, TC_SMEM_BYTES, s>>>(d_tiles, d_cta_begin, d_segs, A, B, C, conjA, nullptr, nullptr);
  ++*lc;
}

}  // namespace fh
