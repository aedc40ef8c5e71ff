// Segmented grouped complex128 GEMM (SURVEY 8(a) rows H1-H5, H8 merge, H10 norm environments):
//     C_o (M x N) = sum_{t in seg(o)} alpha_t * op(A_t) (M x K_t) * op(B_t) (K_t x N),  alpha_t real.
//
// sm_100a has exactly one FP64 tensor-core shape, DMMA.8x8x4 (mma.sync.m8n8k4.f64; tcgen05 has no
// f64 kind), issued at one instruction per 16 cycles per SM sub-partition -- a single warp with two
// independent accumulators already saturates it ("DMMA issue model").  The FP64 pipe is
// therefore never limited by shared-memory or L2 bandwidth on this workload but by everything that
// keeps a warp from issuing DMMAs: tile-shape padding, CTA-wide barriers, pipeline fill and drain.
// The kernel is built around that:
//   * the unit of work is one WARP computing an (8 mt) x (8 nt) sub-tile of one output block over the
//     whole concatenated K of that block (mt * nt <= 16 accumulator sub-tiles in registers); units
//     are cut per block by the host so that only the last 8-row / 8-column sliver is padded;
//   * no CTA-level tile, no __syncthreads: each warp streams its own operand fragments with
//     cp.async (LDGSTS, 16 B per lane, zero-filled beyond a segment's K) into a warp-private
//     shared-memory ring and reads them back with conflict-free LDS.128 -- every lane reads exactly
//     the bytes it copied, so the ring needs no intra-warp synchronisation either;
//   * one unit per one-warp CTA, units sorted heaviest first: the hardware CTA scheduler is the
//     (greedy, longest-processing-time-first) load balancer;
//   * four real DMMAs per complex product, the recoupling coefficient alpha folded into the A
//     fragment (two DMULs per fragment), conjugation folded into the sign of alpha;
//   * outputs are never shared between warps and the k order is fixed by the task list: results are
//     run-to-run bit-identical.
#include "fh_internal.hpp"

namespace fh {

namespace {

__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c[0]), "+d"(c[1])
               : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(uint32_t smem_addr, const void* gptr, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_addr), "l"(gptr), "r"(src_bytes));
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ cplx lds_c(uint32_t addr) {
  cplx v;
  asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  return v;
}

constexpr int RING_DEPTH = 3;     // cp.async stages in flight per warp
constexpr int MAX_FRAGS = 10;     // mt + nt <= 10 for every shape with mt * nt <= 16, mt, nt <= 8
constexpr int RING_BYTES = RING_DEPTH * MAX_FRAGS * 512;

// Producer side of one unit: walks the k-steps of all segments and issues the cp.asyncs of one
// step (mt A fragments + nt B fragments, 16 B per lane each) into a ring stage.
// Fragment layout of DMMA.8x8x4: lane l holds A[row l/4][k l%4] and B[k l%4][col l/4].
template <int MT, int NT>
struct Producer {
  const GemmSeg* segs;
  const cplx *Abase, *Bbase;
  int si, se;
  int s, nfull, nst, K;
  int mi[MT], nj[NT];
  int kq;
  const cplx* pa[MT];
  const cplx* pb[NT];
  int64_t dA, dB;
  int a_sk, b_sk;
  bool done;
  // descriptor of segment si + 1, loaded one segment ahead so that the switch never waits on L2
  int64_t n_a_off, n_b_off;
  int n_K, n_a_sm, n_a_sk, n_b_sk, n_b_sn;

  __device__ __forceinline__ void setup(int64_t a_off, int64_t b_off, int K_, int a_sm, int a_sk_, int b_sk_,
                                        int b_sn) {
    K = K_;
    nfull = K >> 2;
    nst = (K + 3) >> 2;
    s = 0;
    a_sk = a_sk_;
    b_sk = b_sk_;
    const cplx* A0 = Abase + a_off + (int64_t)kq * a_sk_;
    const cplx* B0 = Bbase + b_off + (int64_t)kq * b_sk_;
#pragma unroll
    for (int i = 0; i < MT; ++i) pa[i] = A0 + (int64_t)mi[i] * a_sm;
#pragma unroll
    for (int j = 0; j < NT; ++j) pb[j] = B0 + (int64_t)nj[j] * b_sn;
    dA = 4 * (int64_t)a_sk_;
    dB = 4 * (int64_t)b_sk_;
  }
  __device__ __forceinline__ void prefetch_next() {
    const GemmSeg* np = segs + min(si + 1, se - 1);
    n_a_off = np->a_off;
    n_b_off = np->b_off;
    n_K = np->K;
    n_a_sm = np->a_sm;
    n_a_sk = np->a_sk;
    n_b_sk = np->b_sk;
    n_b_sn = np->b_sn;
  }
  __device__ __forceinline__ void init(const GemmSeg* segs_, const GemmUnit& u, const cplx* A, const cplx* B,
                                       int lane) {
    segs = segs_;
    Abase = A;
    Bbase = B;
    si = u.seg_begin;
    se = u.seg_end;
    kq = lane & 3;
    done = false;
    const int r = lane >> 2;
    // rows / columns beyond the block edge re-read the last valid one: they only feed accumulator
    // rows / columns that are never stored
#pragma unroll
    for (int i = 0; i < MT; ++i) mi[i] = min(u.m0 + 8 * i + r, u.M - 1);
#pragma unroll
    for (int j = 0; j < NT; ++j) nj[j] = min(u.n0 + 8 * j + r, u.N - 1);
    setup(u.first.a_off, u.first.b_off, u.first.K, u.first.a_sm, u.first.a_sk, u.first.b_sk, u.first.b_sn);
    prefetch_next();
  }
  __device__ __forceinline__ void issue(uint32_t dst) {
    if (!done) {
      if (s < nfull) {
#pragma unroll
        for (int i = 0; i < MT; ++i) {
          cp_async16(dst + i * 512, pa[i], 16);
          pa[i] += dA;
        }
#pragma unroll
        for (int j = 0; j < NT; ++j) {
          cp_async16(dst + (MT + j) * 512, pb[j], 16);
          pb[j] += dB;
        }
      } else {
        // ragged k tail of the segment: lanes with k >= K copy nothing and get zeros
        const int k = 4 * nfull + kq;
        const int back = k < K ? 0 : k - (K - 1);
        const int sz = k < K ? 16 : 0;
#pragma unroll
        for (int i = 0; i < MT; ++i) cp_async16(dst + i * 512, pa[i] - (int64_t)back * a_sk, sz);
#pragma unroll
        for (int j = 0; j < NT; ++j) cp_async16(dst + (MT + j) * 512, pb[j] - (int64_t)back * b_sk, sz);
      }
      ++s;
      if (s == nst) {
        ++si;
        if (si < se) {
          setup(n_a_off, n_b_off, n_K, n_a_sm, n_a_sk, n_b_sk, n_b_sn);
          prefetch_next();
        } else {
          done = true;
        }
      }
    }
    cp_commit();
  }
};

template <int MT, int NT>
__device__ __noinline__ void run_unit(const GemmUnit& u, const GemmSeg* __restrict__ segs,
                                      const cplx* __restrict__ A, const cplx* __restrict__ B,
                                      cplx* __restrict__ C, int lane, double conj_sign, uint32_t ring) {
  constexpr int D = RING_DEPTH;
  constexpr int STAGE_BYTES = (MT + NT) * 512;
  double cre[MT][NT][2], cim[MT][NT][2];
#pragma unroll
  for (int i = 0; i < MT; ++i)
#pragma unroll
    for (int j = 0; j < NT; ++j) cre[i][j][0] = cre[i][j][1] = cim[i][j][0] = cim[i][j][1] = 0.0;
  const int total = u.steps;
  if (total > 0) {
    Producer<MT, NT> P;
    P.init(segs, u, A, B, lane);
    const uint32_t lane_ring = ring + lane * 16;
#pragma unroll 1
    for (int d = 0; d < D - 1; ++d) P.issue(lane_ring + d * STAGE_BYTES);
    // consumer-side walk over the segments for alpha, one segment of lookahead
    int csi = u.seg_begin;
    const int cse = u.seg_end;
    int cleft = (u.first.K + 3) >> 2;
    double alpha = u.first.alpha;
    int nK = segs[min(csi + 1, cse - 1)].K;
    double nalpha = segs[min(csi + 1, cse - 1)].alpha;
    int rd = 0, wr = D - 1;
#pragma unroll 1
    for (int t = 0; t < total; ++t) {
      cp_wait<D - 2>();
      const uint32_t src = lane_ring + rd * STAGE_BYTES;
      double ar[MT], ai[MT];
      const double als = alpha * conj_sign;
#pragma unroll
      for (int i = 0; i < MT; ++i) {
        const cplx v = lds_c(src + i * 512);
        ar[i] = alpha * v.x;
        ai[i] = als * v.y;
      }
      cplx b[NT];
#pragma unroll
      for (int j = 0; j < NT; ++j) b[j] = lds_c(src + (MT + j) * 512);
      P.issue(lane_ring + wr * STAGE_BYTES);
      rd = rd + 1 == D ? 0 : rd + 1;
      wr = wr + 1 == D ? 0 : wr + 1;
      // (ar + i ai)(br + i bi): four real DMMAs per 8x8 sub-tile, ordered so that consecutive
      // DMMAs never touch the same accumulator
#pragma unroll
      for (int j = 0; j < NT; ++j)
#pragma unroll
        for (int i = 0; i < MT; ++i) dmma884(cre[i][j], ar[i], b[j].x);
#pragma unroll
      for (int j = 0; j < NT; ++j)
#pragma unroll
        for (int i = 0; i < MT; ++i) dmma884(cim[i][j], ar[i], b[j].y);
#pragma unroll
      for (int j = 0; j < NT; ++j)
#pragma unroll
        for (int i = 0; i < MT; ++i) dmma884(cre[i][j], -ai[i], b[j].y);
#pragma unroll
      for (int j = 0; j < NT; ++j)
#pragma unroll
        for (int i = 0; i < MT; ++i) dmma884(cim[i][j], ai[i], b[j].x);
      if (--cleft == 0) {
        ++csi;
        cleft = (nK + 3) >> 2;
        alpha = nalpha;
        const GemmSeg* np = segs + min(csi + 1, cse - 1);
        nK = np->K;
        nalpha = np->alpha;
      }
    }
    cp_wait<0>();
  }
  // epilogue: lane holds C[row lane/4][cols 2 (lane%4), 2 (lane%4) + 1] of every sub-tile
  const int er = lane >> 2, ec = (lane & 3) * 2;
  cplx* gC = C + u.c_off;
#pragma unroll
  for (int i = 0; i < MT; ++i) {
    const int r = u.m0 + 8 * i + er;
    if (r < u.M) {
#pragma unroll
      for (int j = 0; j < NT; ++j) {
        const int c = u.n0 + 8 * j + ec;
        cplx* p = gC + (int64_t)r * u.ldc + c;
        if (c < u.N) p[0] = make_double2(cre[i][j][0], cim[i][j][0]);
        if (c + 1 < u.N) p[1] = make_double2(cre[i][j][1], cim[i][j][1]);
      }
    }
  }
}

#define FH_FOR_SHAPES(X)                                                                                   \
  X(1, 1) X(1, 2) X(1, 3) X(1, 4) X(1, 5) X(1, 6) X(1, 7) X(1, 8) X(2, 1) X(2, 2) X(2, 3) X(2, 4) X(2, 5)  \
  X(2, 6) X(2, 7) X(2, 8) X(3, 1) X(3, 2) X(3, 3) X(3, 4) X(3, 5) X(4, 1) X(4, 2) X(4, 3) X(4, 4) X(5, 1)  \
  X(5, 2) X(5, 3) X(6, 1) X(6, 2) X(7, 1) X(7, 2) X(8, 1) X(8, 2)

__global__ void __launch_bounds__(32) grouped_zgemm_kernel(const GemmUnit* __restrict__ units, int nunits,
                                                           const GemmSeg* __restrict__ segs,
                                                           const cplx* __restrict__ A, const cplx* __restrict__ B,
                                                           cplx* __restrict__ C, int conjA) {
  __shared__ __align__(128) unsigned char ring_smem[RING_BYTES];
  const int lane = threadIdx.x;
  const int ui = blockIdx.x;
  if (ui >= nunits) return;
  const GemmUnit u = units[ui];
  const uint32_t ring = (uint32_t)__cvta_generic_to_shared(ring_smem);
  const double cs = conjA ? -1.0 : 1.0;
  switch (u.shape) {
#define FH_CASE(MT, NT)                                    \
  case MT * 16 + NT:                                       \
    run_unit<MT, NT>(u, segs, A, B, C, lane, cs, ring);    \
    break;
    FH_FOR_SHAPES(FH_CASE)
#undef FH_CASE
    default:
      break;
  }
}

}  // namespace

void launch_grouped_gemm(const Stage& st, const cplx* A, const cplx* B, cplx* C, cudaStream_t s, int64_t* lc) {
  const int n = (int)st.units.size();
  if (n == 0) return;
  grouped_zgemm_kernel<<<n, 32, 0, s>>>(st.d_units, n, st.d_segs, A, B, C, st.opA != OPA_N ? 1 : 0);
  ++*lc;
}

}  // namespace fh
