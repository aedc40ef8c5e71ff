// Hand-written sm_100a kernels of the hot path:
//   * grouped_zgemm_kernel: segmented grouped complex128 GEMM over a tile queue,
//       C_o (M x N) = sum_{t in seg(o)} alpha_t * op(A_t) (M x K_t) * op(B_t) (K_t x N)
//     FP64 tensor-core path: mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4, the only FP64 MMA shape
//     sm_100a has; tcgen05 has no f64 kind), four real DMMAs per complex product, operands staged
//     through a multi-stage cp.async (LDGSTS) ring with zero-filled ragged edges, the real
//     recoupling coefficient alpha fused into the A-fragment load, padding sub-tiles skipped.
//   * weighted dot / axpy / linear-combination kernels for the Lanczos recurrences (HBM-bound).
//   * block gather/scatter with scaling for pack/unpack around the block-wise SVD (HBM-bound).
// Outputs are never shared between CTAs and reductions run in a fixed order: results are
// run-to-run bit-identical.
#include "fh_internal.hpp"

namespace fh {

// ------------------------------------------------------------------------------------------
// PTX wrappers
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
      : "+d"(c0), "+d"(c1)
      : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(uint32_t smem_addr, const void* gptr, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_addr), "l"(gptr), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N));
}

// ------------------------------------------------------------------------------------------
// Segmented grouped ZGEMM
// ------------------------------------------------------------------------------------------
// Shared-memory tile layouts (BK = 8 complex per pipeline stage):
//   K-minor (operand stored with k contiguous: A for OPA_N/OPA_C, B for OPB_T):
//       [BK/4][ROWS][4] complex  -> a fragment load (row = lane/4, k = lane%4) of a quarter
//       warp touches 128 contiguous bytes: conflict-free without padding.
//   K-major (operand stored with the m / n index contiguous: A for OPA_H, B for OPB_N):
//       [BK][COLS + 2] complex   -> row pitch = 32 B mod 128: the 4 k-rows of a quarter warp
//       land in distinct 32-byte bank groups: conflict-free.
constexpr int BK = 8;

template <int ROWS, bool KMINOR>
struct TileLayout {
  static constexpr int elems = KMINOR ? ROWS * BK : BK * (ROWS + 2);
  // element index of (row r, k)
  __device__ static __forceinline__ int at(int r, int k) {
    return KMINOR ? (((k >> 2) * ROWS + r) << 2) + (k & 3) : k * (ROWS + 2) + r;
  }
};

template <int BM, int BN, int WARPS_M, int WARPS_N, int OPA, int OPB, int STAGES>
__global__ void __launch_bounds__(WARPS_M* WARPS_N * 32)
    grouped_zgemm_kernel(const GemmTile* __restrict__ tiles, const GemmOut* __restrict__ outs,
                         const GemmSeg* __restrict__ segs, const cplx* __restrict__ Abase,
                         const cplx* __restrict__ Bbase, cplx* __restrict__ Cbase) {
  constexpr int NT = WARPS_M * WARPS_N * 32;
  constexpr int WM = BM / WARPS_M, WN = BN / WARPS_N;
  constexpr int MT = WM / 8, NTL = WN / 8;
  constexpr bool A_KMINOR = (OPA != OPA_H);
  constexpr bool B_KMINOR = (OPB == OPB_T);
  typedef TileLayout<BM, A_KMINOR> LA;
  typedef TileLayout<BN, B_KMINOR> LB;
  constexpr int STAGE_ELEMS = LA::elems + LB::elems;

  extern __shared__ __align__(128) unsigned char smem_raw[];
  cplx* smem = reinterpret_cast<cplx*>(smem_raw);

  const GemmTile tile = tiles[blockIdx.x];
  const GemmOut out = outs[tile.out];
  const int M = out.M, N = out.N;
  const int m0 = tile.m0, n0 = tile.n0;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm0 = (warp / WARPS_N) * WM, wn0 = (warp % WARPS_N) * WN;
  const int mrem = M - m0, nrem = N - n0;  // valid rows / cols in this tile (may exceed BM / BN)

  // number of 8x8 sub-tiles of this warp that hold real data (edge skipping, warp-uniform)
  int mt_valid = (mrem - wm0 + 7) >> 3;
  mt_valid = mt_valid < 0 ? 0 : (mt_valid > MT ? MT : mt_valid);
  int nt_valid = (nrem - wn0 + 7) >> 3;
  nt_valid = nt_valid < 0 ? 0 : (nt_valid > NTL ? NTL : nt_valid);

  double acc_re[MT][NTL][2], acc_im[MT][NTL][2];
#pragma unroll
  for (int i = 0; i < MT; ++i)
#pragma unroll
    for (int j = 0; j < NTL; ++j) acc_re[i][j][0] = acc_re[i][j][1] = acc_im[i][j][0] = acc_im[i][j][1] = 0.0;

  // ---- chunk iterators: a chunk is BK consecutive k of one segment
  int ld_seg = out.seg_begin, ld_k0 = 0;
  int cp_seg = out.seg_begin, cp_k0 = 0;
  const int seg_end = out.seg_end;

  auto load_chunk = [&](int stage) {
    if (ld_seg < seg_end) {
      const GemmSeg sg = segs[ld_seg];
      cplx* sA = smem + stage * STAGE_ELEMS;
      cplx* sB = sA + LA::elems;
      const cplx* gA = Abase + sg.a_off;
      const cplx* gB = Bbase + sg.b_off;
      const int kleft = sg.K - ld_k0;
      // A tile: BM rows x BK
#pragma unroll
      for (int idx = tid; idx < BM * BK; idx += NT) {
        int r, k;
        if (A_KMINOR) { r = idx / BK; k = idx % BK; } else { k = idx / BM; r = idx % BM; }
        const bool ok = (r < mrem) && (k < kleft);
        const cplx* src = gA;
        if (ok) src = A_KMINOR ? gA + (int64_t)(m0 + r) * sg.lda + (ld_k0 + k)
                               : gA + (int64_t)(ld_k0 + k) * sg.lda + (m0 + r);
        cp_async16((uint32_t)__cvta_generic_to_shared(sA + LA::at(r, k)), src, ok ? 16 : 0);
      }
      // B tile: BK x BN cols
#pragma unroll
      for (int idx = tid; idx < BN * BK; idx += NT) {
        int c, k;
        if (B_KMINOR) { c = idx / BK; k = idx % BK; } else { k = idx / BN; c = idx % BN; }
        const bool ok = (c < nrem) && (k < kleft);
        const cplx* src = gB;
        if (ok) src = B_KMINOR ? gB + (int64_t)(n0 + c) * sg.ldb + (ld_k0 + k)
                               : gB + (int64_t)(ld_k0 + k) * sg.ldb + (n0 + c);
        cp_async16((uint32_t)__cvta_generic_to_shared(sB + LB::at(c, k)), src, ok ? 16 : 0);
      }
      ld_k0 += BK;
      if (ld_k0 >= sg.K) { ld_k0 = 0; ++ld_seg; }
    }
    cp_async_commit();
  };

#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s) load_chunk(s);

  int stage = 0;
  while (cp_seg < seg_end) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    {
      int ld_stage = stage + STAGES - 1;
      if (ld_stage >= STAGES) ld_stage -= STAGES;
      load_chunk(ld_stage);
    }
    const GemmSeg sg = segs[cp_seg];
    const double alpha = sg.alpha;
    const int kvalid = sg.K - cp_k0;  // > 0
    const int nk4 = kvalid >= BK ? BK / 4 : (kvalid + 3) >> 2;
    const cplx* sA = smem + stage * STAGE_ELEMS;
    const cplx* sB = sA + LA::elems;
    const int fr = lane >> 2, fk = lane & 3;
#pragma unroll
    for (int kk = 0; kk < BK / 4; ++kk) {
      if (kk < nk4) {
        double a_re[MT], a_im[MT], a_nim[MT];
#pragma unroll
        for (int i = 0; i < MT; ++i) {
          if (i < mt_valid) {
            const cplx v = sA[LA::at(wm0 + i * 8 + fr, kk * 4 + fk)];
            a_re[i] = alpha * v.x;
            const double im = alpha * v.y;
            a_im[i] = (OPA == OPA_N) ? im : -im;  // conj for OPA_C / OPA_H
            a_nim[i] = -a_im[i];
          }
        }
#pragma unroll
        for (int j = 0; j < NTL; ++j) {
          if (j < nt_valid) {
            const cplx b = sB[LB::at(wn0 + j * 8 + fr, kk * 4 + fk)];
#pragma unroll
            for (int i = 0; i < MT; ++i) {
              if (i < mt_valid) {
                dmma884(acc_re[i][j][0], acc_re[i][j][1], a_re[i], b.x);
                dmma884(acc_im[i][j][0], acc_im[i][j][1], a_re[i], b.y);
                dmma884(acc_re[i][j][0], acc_re[i][j][1], a_nim[i], b.y);
                dmma884(acc_im[i][j][0], acc_im[i][j][1], a_im[i], b.x);
              }
            }
          }
        }
      }
    }
    cp_k0 += BK;
    if (cp_k0 >= sg.K) { cp_k0 = 0; ++cp_seg; }
    stage = stage + 1 == STAGES ? 0 : stage + 1;
  }
  cp_async_wait<0>();

  // ---- epilogue: thread holds C[row = lane/4][col = (lane%4)*2 + {0,1}] of every sub-tile
  cplx* gC = Cbase + out.c_off;
  const int er = lane >> 2, ec = (lane & 3) * 2;
#pragma unroll
  for (int i = 0; i < MT; ++i) {
    const int r = m0 + wm0 + i * 8 + er;
    if (i < mt_valid && r < M) {
#pragma unroll
      for (int j = 0; j < NTL; ++j) {
        const int c = n0 + wn0 + j * 8 + ec;
        if (j < nt_valid) {
          cplx* p = gC + (int64_t)r * N + c;
          if (c < N) p[0] = make_double2(acc_re[i][j][0], acc_im[i][j][0]);
          if (c + 1 < N) p[1] = make_double2(acc_re[i][j][1], acc_im[i][j][1]);
        }
      }
    }
  }
}

template <int BM, int BN, int WARPS_M, int WARPS_N, int STAGES>
static void launch_variant(const Stage& st, const GemmTile* d_tiles, int ntiles, const cplx* A, const cplx* B,
                           cplx* C, cudaStream_t s) {
  if (ntiles == 0) return;
  constexpr int NT = WARPS_M * WARPS_N * 32;
#define FH_LAUNCH(OA, OB)                                                                          \
  {                                                                                                \
    constexpr bool AK = (OA != OPA_H);                                                             \
    constexpr bool BKM = (OB == OPB_T);                                                            \
    constexpr size_t smem = (size_t)STAGES * (TileLayout<BM, AK>::elems + TileLayout<BN, BKM>::elems) * sizeof(cplx); \
    auto kern = grouped_zgemm_kernel<BM, BN, WARPS_M, WARPS_N, OA, OB, STAGES>;                    \
    static bool attr_done = false;                                                                 \
    if (!attr_done) {                                                                              \
      cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);          \
      attr_done = true;                                                                            \
    }                                                                                              \
    kern<<<ntiles, NT, smem, s>>>(d_tiles, st.d_outs, st.d_segs, A, B, C);                          \
  }
  if (st.opA == OPA_N && st.opB == OPB_N) FH_LAUNCH(OPA_N, OPB_N)
  else if (st.opA == OPA_N && st.opB == OPB_T) FH_LAUNCH(OPA_N, OPB_T)
  else if (st.opA == OPA_C && st.opB == OPB_N) FH_LAUNCH(OPA_C, OPB_N)
  else if (st.opA == OPA_H && st.opB == OPB_N) FH_LAUNCH(OPA_H, OPB_N)
#undef FH_LAUNCH
}

void launch_grouped_gemm(const Stage& st, const cplx* A, const cplx* B, cplx* C, cudaStream_t s,
                         int64_t* lc) {
  if (!st.tiles64.empty()) {
    launch_variant<64, 64, 2, 2, 4>(st, st.d_tiles64, (int)st.tiles64.size(), A, B, C, s);
    ++*lc;
  }
  if (!st.tiles32.empty()) {
    launch_variant<32, 32, 2, 2, 4>(st, st.d_tiles32, (int)st.tiles32.size(), A, B, C, s);
    ++*lc;
  }
}

// ------------------------------------------------------------------------------------------
// Lanczos vector kernels (H6)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}

// partial[2*chunk + {0,1}] = w_chunk * sum conj(x) y over the chunk (fixed order inside the CTA)
__global__ void __launch_bounds__(256) wdot_partial_kernel(const VecChunk* __restrict__ chunks,
                                                           const cplx* __restrict__ x,
                                                           const cplx* __restrict__ y,
                                                           double* __restrict__ partial) {
  const VecChunk ch = chunks[blockIdx.x];
  const cplx* px = x + ch.start;
  const cplx* py = y + ch.start;
  double re = 0.0, im = 0.0;
  for (int i = threadIdx.x; i < ch.len; i += 256) {
    const cplx a = px[i], b = py[i];
    re += a.x * b.x + a.y * b.y;
    im += a.x * b.y - a.y * b.x;
  }
  __shared__ double sre[8], sim[8];
  re = warp_sum(re);
  im = warp_sum(im);
  if ((threadIdx.x & 31) == 0) { sre[threadIdx.x >> 5] = re; sim[threadIdx.x >> 5] = im; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double r = 0.0, m = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { r += sre[i]; m += sim[i]; }
    partial[2 * blockIdx.x] = (double)ch.w * r;
    partial[2 * blockIdx.x + 1] = (double)ch.w * m;
  }
}

// result[0..1] = sum of partials in index order (one CTA, fixed tree)
__global__ void __launch_bounds__(256) wdot_final_kernel(const double* __restrict__ partial, int n,
                                                         double* __restrict__ result) {
  double re = 0.0, im = 0.0;
  for (int i = threadIdx.x; i < n; i += 256) { re += partial[2 * i]; im += partial[2 * i + 1]; }
  __shared__ double sre[8], sim[8];
  re = warp_sum(re);
  im = warp_sum(im);
  if ((threadIdx.x & 31) == 0) { sre[threadIdx.x >> 5] = re; sim[threadIdx.x >> 5] = im; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double r = 0.0, m = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { r += sre[i]; m += sim[i]; }
    result[0] = r;
    result[1] = m;
  }
}

void launch_wdot(const VecChunk* d_chunks, int nchunks, const cplx* x, const cplx* y, double* d_partial,
                 double* d_result, cudaStream_t s, int64_t* lc) {
  wdot_partial_kernel<<<nchunks, 256, 0, s>>>(d_chunks, x, y, d_partial);
  ++*lc;
  if (d_result) {
    wdot_final_kernel<<<1, 256, 0, s>>>(d_partial, nchunks, d_result);
    ++*lc;
  }
}

void launch_block_norms(const VecChunk* d_chunks, int nchunks, const cplx* x, double* d_out, cudaStream_t s,
                        int64_t* lc) {
  wdot_partial_kernel<<<nchunks, 256, 0, s>>>(d_chunks, x, x, d_out);
  ++*lc;
}

__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

__global__ void __launch_bounds__(256) axpy_kernel(int64_t n, cplx a, const cplx* __restrict__ x,
                                                   cplx* __restrict__ y) {
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (int64_t)gridDim.x * 256) {
    const cplx t = cmul(a, x[i]);
    cplx v = y[i];
    v.x += t.x;
    v.y += t.y;
    y[i] = v;
  }
}
__global__ void __launch_bounds__(256) scale_kernel(int64_t n, cplx a, const cplx* __restrict__ x,
                                                    cplx* __restrict__ y) {
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (int64_t)gridDim.x * 256)
    y[i] = cmul(a, x[i]);
}
struct LinCoef {
  cplx c[32];
};
__global__ void __launch_bounds__(256) lincomb_kernel(int64_t n, int m, LinCoef coef, const cplx* __restrict__ V,
                                                      int64_t stride, cplx* __restrict__ y) {
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (int64_t)gridDim.x * 256) {
    double re = 0.0, im = 0.0;
    for (int j = 0; j < m; ++j) {
      const cplx t = cmul(coef.c[j], V[j * stride + i]);
      re += t.x;
      im += t.y;
    }
    y[i] = make_double2(re, im);
  }
}
__global__ void __launch_bounds__(256) zero_kernel(cplx* p, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (int64_t)gridDim.x * 256)
    p[i] = make_double2(0.0, 0.0);
}

static int grid_for(int64_t n) {
  int64_t g = (n + 255) / 256;
  const int64_t cap = 148 * 8;  // 8 CTAs of 256 threads per SM
  return (int)(g < 1 ? 1 : (g > cap ? cap : g));
}
void launch_axpy(int64_t n, cplx a, const cplx* x, cplx* y, cudaStream_t s, int64_t* lc) {
  if (n <= 0) return;
  axpy_kernel<<<grid_for(n), 256, 0, s>>>(n, a, x, y);
  ++*lc;
}
void launch_scale(int64_t n, cplx a, const cplx* x, cplx* y, cudaStream_t s, int64_t* lc) {
  if (n <= 0) return;
  scale_kernel<<<grid_for(n), 256, 0, s>>>(n, a, x, y);
  ++*lc;
}
void launch_lincomb(int64_t n, int m, const cplx* coef_host, const cplx* V, int64_t stride, cplx* y,
                    cudaStream_t s, int64_t* lc) {
  if (n <= 0) return;
  LinCoef c;
  for (int j = 0; j < 32; ++j) c.c[j] = j < m ? coef_host[j] : make_double2(0, 0);
  lincomb_kernel<<<grid_for(n), 256, 0, s>>>(n, m, c, V, stride, y);
  ++*lc;
}
void launch_fill_zero(cplx* p, int64_t n, cudaStream_t s, int64_t* lc) {
  if (n <= 0) return;
  zero_kernel<<<grid_for(n), 256, 0, s>>>(p, n);
  ++*lc;
}

// ------------------------------------------------------------------------------------------
// pack / unpack (H8): scaled block copies between the block-sparse layout and dense matrices
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) copy_blocks_kernel(const CopyBlk* __restrict__ blks,
                                                          const cplx* __restrict__ src, cplx* __restrict__ dst) {
  const CopyBlk b = blks[blockIdx.x];
  const cplx* ps = src + b.src_off;
  cplx* pd = dst + b.dst_off;
  const int64_t total = (int64_t)b.rows * b.cols;
  for (int64_t i = (int64_t)blockIdx.y * 256 + threadIdx.x; i < total; i += (int64_t)gridDim.y * 256) {
    const int r = (int)(i / b.cols), c = (int)(i % b.cols);
    cplx v = ps[(int64_t)r * b.ld_src + c];
    v.x *= b.scale;
    v.y *= b.scale;
    if (b.transpose_dst) pd[(int64_t)c * b.ld_dst + r] = v;
    else pd[(int64_t)r * b.ld_dst + c] = v;
  }
}
void launch_copy_blocks(const CopyBlk* d_blks, int nblk, const cplx* src, cplx* dst, cudaStream_t s,
                        int64_t* lc) {
  if (nblk <= 0) return;
  dim3 grid(nblk, 8);
  copy_blocks_kernel<<<grid, 256, 0, s>>>(d_blks, src, dst);
  ++*lc;
}

// ------------------------------------------------------------------------------------------
// calibration: FP64 tensor-pipe issue peak (roofline denominator, not on the hot path)
// ------------------------------------------------------------------------------------------
constexpr int PEAK_ITERS = 2048, PEAK_ACC = 8;
__global__ void __launch_bounds__(256) dmma_peak_kernel(double* out) {
  double c[PEAK_ACC][2];
#pragma unroll
  for (int i = 0; i < PEAK_ACC; ++i) c[i][0] = c[i][1] = threadIdx.x * 1e-9 + i;
  const double a = 1.0 + threadIdx.x * 1e-7, b = 1.0 - threadIdx.x * 1e-7;
  for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
    for (int i = 0; i < PEAK_ACC; ++i) dmma884(c[i][0], c[i][1], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < PEAK_ACC; ++i) s += c[i][0] + c[i][1];
  out[blockIdx.x * 256 + threadIdx.x] = s;
}
double launch_dmma_peak(double* scratch, cudaStream_t s, int64_t* lc) {
  const int ctas = 148 * 4;
  dmma_peak_kernel<<<ctas, 256, 0, s>>>(scratch);
  ++*lc;
  return 2.0 * 256.0 * PEAK_ITERS * PEAK_ACC * 8.0 * ctas;  // 8 warps x 256 FMA per DMMA.8x8x4
}

}  // namespace fh
