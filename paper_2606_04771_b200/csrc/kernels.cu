// Hand-written sm_100a kernels of the bandwidth-bound part of the hot path:
//   * weighted dot / axpy / linear-combination kernels for the Lanczos recurrences;
//   * block gather/scatter with scaling for pack/unpack around the block-wise SVD;
//   * the DMMA issue-peak calibration kernel (roofline denominator).
// The segmented grouped ZGEMM (H1-H5) lives in zgemm.cu.
// Reductions run in a fixed order: results are run-to-run bit-identical.
#include "fh_internal.hpp"

#include <cstdlib>

namespace fh {

bool pdl_enabled(int role) { return (PDL_DEFAULT_MASK & role) != 0; }

// ------------------------------------------------------------------------------------------
// PTX wrappers
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
      : "+d"(c0), "+d"(c1)
      : "d"(a), "d"(b));
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

// The CTA that retires last (atomicInc on a counter that wraps back to zero) adds the partials in index order
// with the tree of wdot_final_kernel: one launch instead of two, same bits whichever CTA happens to be last.
__device__ __forceinline__ void finish_in_last_cta(const double* __restrict__ partial, int n, double* __restrict__ result,
                                                   unsigned* __restrict__ counter) {
  __shared__ bool is_last;
  __shared__ double fre[8], fim[8];
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) is_last = atomicInc(counter, gridDim.x - 1) == gridDim.x - 1;
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  double re = 0.0, im = 0.0;
  for (int i = threadIdx.x; i < n; i += 256) {
    re += __ldcg(partial + 2 * i);
    im += __ldcg(partial + 2 * i + 1);
  }
  re = warp_sum(re);
  im = warp_sum(im);
  if ((threadIdx.x & 31) == 0) { fre[threadIdx.x >> 5] = re; fim[threadIdx.x >> 5] = im; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double r = 0.0, m = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { r += fre[i]; m += fim[i]; }
    result[0] = r;
    result[1] = m;
  }
}

// <x, y> in one launch (partials + last-CTA sum)
__global__ void __launch_bounds__(256) wdot_fused_kernel(const VecChunk* __restrict__ chunks, const cplx* __restrict__ x,
                                                         const cplx* __restrict__ y, double* __restrict__ partial,
                                                         double* __restrict__ result, unsigned* __restrict__ counter) {
  pdl_launch_dependents();
  const VecChunk ch = chunks[blockIdx.x];
  pdl_wait();
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
  finish_in_last_cta(partial, gridDim.x, result, counter);
}

// Lanczos three-term update on UNNORMALISED Krylov vectors, and the norm of its result, in one launch.
// The recurrence keeps u_j = b_j v_j (b_0 = 1, b_j = beta_{j-1} = |u_j|) instead of v_j, so that no separate
// normalisation pass is needed:  with w = H u_j and a_raw = <u_j, w>,
//   alpha_j = a_raw / b_j^2,   u_{j+1} = (w - alpha_j u_j) / b_j - (b_j / b_{j-1}) u_{j-1},   result = <u_{j+1}, u_{j+1}>
// (= beta_j^2).  b_j^2 and b_{j-1}^2 are the results of the two previous updates (NULL = 1).  A norm below tol
// (happy breakdown) makes its reciprocal 0, as the normalisation pass did: everything stays finite and the host
// truncates the Krylov space there.
__global__ void __launch_bounds__(256) lanczos_update_kernel(const VecChunk* __restrict__ chunks,
                                                             const double* __restrict__ a_raw,
                                                             const double* __restrict__ bj2,
                                                             const double* __restrict__ bjm2, double tol,
                                                             const cplx* __restrict__ vj, const cplx* __restrict__ vprev,
                                                             cplx* __restrict__ w, double* __restrict__ partial,
                                                             double* __restrict__ result, unsigned* __restrict__ counter) {
  pdl_launch_dependents();
  const VecChunk ch = chunks[blockIdx.x];
  pdl_wait();
  double bj = 1.0, f = 1.0;
  if (bj2) {
    bj = sqrt(fmax(bj2[0], 0.0));
    f = (bj < tol || bj == 0.0) ? 0.0 : 1.0 / bj;
  }
  const double a = -(a_raw[0] * f * f) * f;
  double b = 0.0;
  if (vprev) {
    double fm = 1.0;
    if (bjm2) {
      const double bm = sqrt(fmax(bjm2[0], 0.0));
      fm = (bm < tol || bm == 0.0) ? 0.0 : 1.0 / bm;
    }
    b = -bj * fm;
  }
  const cplx* pv = vj + ch.start;
  const cplx* pp = vprev ? vprev + ch.start : nullptr;
  cplx* pw = w + ch.start;
  double re = 0.0;
  for (int i = threadIdx.x; i < ch.len; i += 256) {
    const cplx xv = pv[i];
    cplx v = pw[i];
    v.x = f * v.x + a * xv.x;
    v.y = f * v.y + a * xv.y;
    if (pp) {
      const cplx yv = pp[i];
      v.x += b * yv.x;
      v.y += b * yv.y;
    }
    pw[i] = v;
    re += v.x * v.x + v.y * v.y;
  }
  __shared__ double sre[8];
  re = warp_sum(re);
  if ((threadIdx.x & 31) == 0) sre[threadIdx.x >> 5] = re;
  __syncthreads();
  if (threadIdx.x == 0) {
    double r = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) r += sre[i];
    partial[2 * blockIdx.x] = (double)ch.w * r;
    partial[2 * blockIdx.x + 1] = 0.0;
  }
  finish_in_last_cta(partial, gridDim.x, result, counter);
}

void launch_wdot_fused(const VecChunk* d_chunks, int nchunks, const cplx* x, const cplx* y, double* d_partial,
                       double* d_result, unsigned* d_counter, cudaStream_t s, int64_t* lc) {
  launch_pdl(PDL_WDOT, wdot_fused_kernel, nchunks, 256, s, d_chunks, x, y, d_partial, d_result, d_counter);
  ++*lc;
}
void launch_lanczos_update(const VecChunk* d_chunks, int nchunks, const double* d_a_raw, const double* d_bj2,
                           const double* d_bjm2, double tol, const cplx* vj, const cplx* vprev, cplx* w,
                           double* d_partial, double* d_result, unsigned* d_counter, cudaStream_t s, int64_t* lc) {
  launch_pdl(PDL_UPDATE, lanczos_update_kernel, nchunks, 256, s, d_chunks, d_a_raw, d_bj2, d_bjm2, tol, vj, vprev, w,
             d_partial, d_result, d_counter);
  ++*lc;
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
// Device-scalar variant for the Lanczos recurrence (no host round trip inside the iteration):
// y = x / sqrt(norm2[0]); beta_out[0] = sqrt(norm2[0]).  Below tol the direction is dropped (y = 0):
// the host sees beta < tol afterwards and truncates the Krylov space there (happy breakdown).
__global__ void __launch_bounds__(256) scale_rsqrt_dev_kernel(int64_t n, const double* __restrict__ norm2, double tol,
                                                              const cplx* __restrict__ x, cplx* __restrict__ y,
                                                              double* __restrict__ beta_out) {
  pdl_launch_dependents();
  pdl_wait();
  const double b = sqrt(fmax(norm2[0], 0.0));
  const double f = (b < tol || b == 0.0) ? 0.0 : 1.0 / b;
  if (blockIdx.x == 0 && threadIdx.x == 0 && beta_out) beta_out[0] = b;
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (int64_t)gridDim.x * 256) {
    const cplx xv = x[i];
    y[i] = make_double2(f * xv.x, f * xv.y);
  }
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
void launch_scale_rsqrt_dev(int64_t n, const double* d_norm2, double tol, const cplx* x, cplx* y, double* d_beta,
                            cudaStream_t s, int64_t* lc) {
  if (n <= 0) return;
  launch_pdl(PDL_SCALE, scale_rsqrt_dev_kernel, grid_for(n), 256, s, n, d_norm2, tol, x, y, d_beta);
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
  if (!b.transpose_dst) {
    const int64_t total = (int64_t)b.rows * b.cols;
    for (int64_t i = (int64_t)blockIdx.y * 256 + threadIdx.x; i < total; i += (int64_t)gridDim.y * 256) {
      const int r = (int)(i / b.cols), c = (int)(i % b.cols);
      cplx v = ps[(int64_t)r * b.ld_src + c];
      v.x *= b.scale;
      v.y *= b.scale;
      pd[(int64_t)r * b.ld_dst + c] = v;
    }
    return;
  }
  // transposing copy: 32 x 32 tiles through shared memory so that both the reads (rows of src)
  // and the writes (rows of dst) are contiguous 512-byte runs
  __shared__ cplx tile[32][33];
  const int tr = (b.rows + 31) >> 5, tc = (b.cols + 31) >> 5;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;  // 32 x 8 threads
  for (int t = blockIdx.y; t < tr * tc; t += gridDim.y) {
    const int r0 = (t / tc) << 5, c0 = (t % tc) << 5;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int r = r0 + ty + 8 * k, c = c0 + tx;
      if (r < b.rows && c < b.cols) {
        cplx v = ps[(int64_t)r * b.ld_src + c];
        v.x *= b.scale;
        v.y *= b.scale;
        tile[ty + 8 * k][tx] = v;
      }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int c = c0 + ty + 8 * k, r = r0 + tx;  // dst row = src column
      if (r < b.rows && c < b.cols) pd[(int64_t)c * b.ld_dst + r] = tile[tx][ty + 8 * k];
    }
    __syncthreads();
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
