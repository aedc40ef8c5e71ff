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

constexpr int RING_DEPTH = 4;     // cp.async ring stages per warp (power of two)
constexpr int MAX_FRAGS = 10;     // mt + nt <= 10 for every shape with mt * nt <= 16, mt, nt <= 8
constexpr int RING_BYTES = RING_DEPTH * MAX_FRAGS * 512;

// One unit = the flattened k-step sequence of all segments of an output block.  Step t is consumed
// (LDS + 4 mt nt DMMAs) while step t + D - 1 is being copied.  The sequence is cut into chunks inside
// which neither the consumer nor the producer (D - 1 steps ahead) changes segment and the producer
// copies only full 4-wide k-steps: the chunk loop carries no bookkeeping at all (per k-step: mt + nt
// LDGSTS with their pointer updates, mt + nt LDS.128, 2 mt DMUL, one wait, one commit).  Ragged k
// tails, segment switches and the drain run through the slow path, one step at a time.
// Fragment layout of DMMA.8x8x4: lane l holds A[row l/4][k l%4] and B[k l%4][col l/4].
// Rows / columns beyond the block edge re-read the last valid one: they only feed accumulator rows /
// columns that are never stored.  Lanes with k >= K copy zero bytes and get zeros (cp.async zero fill).
#define P_SETUP(AOFF, BOFF, KK, ASM, ASK, BSK, BSN)                         \
  {                                                                         \
    p_K = (KK);                                                             \
    p_left = (p_K + 3) >> 2;                                                \
    p_ask = (ASK);                                                          \
    p_bsk = (BSK);                                                          \
    const cplx* A0 = A + (AOFF) + (int64_t)kq * p_ask;                      \
    const cplx* B0 = B + (BOFF) + (int64_t)kq * p_bsk;                      \
    const int asm_ = (ASM), bsn_ = (BSN);                                   \
    _Pragma("unroll") for (int i = 0; i < MT; ++i) pa[i] = A0 + (int64_t)mi[i] * asm_; \
    _Pragma("unroll") for (int j = 0; j < NT; ++j) pb[j] = B0 + (int64_t)nj[j] * bsn_; \
    dA = 4 * (int64_t)p_ask;                                                \
    dB = 4 * (int64_t)p_bsk;                                                \
  }
#define P_STEP_SLOW(DST)                                                                         \
  {                                                                                              \
    const uint32_t dst_ = (DST);                                                                 \
    if (p_issued < total) {                                                                      \
      const int k = 4 * (((p_K + 3) >> 2) - p_left) + kq;                                        \
      const int back = k < p_K ? 0 : k - (p_K - 1);                                              \
      const int sz = k < p_K ? 16 : 0;                                                           \
      _Pragma("unroll") for (int i = 0; i < MT; ++i) {                                           \
        cp_async16(dst_ + i * 512, pa[i] - (int64_t)back * p_ask, sz);                           \
        pa[i] += dA;                                                                             \
      }                                                                                          \
      _Pragma("unroll") for (int j = 0; j < NT; ++j) {                                           \
        cp_async16(dst_ + (MT + j) * 512, pb[j] - (int64_t)back * p_bsk, sz);                    \
        pb[j] += dB;                                                                             \
      }                                                                                          \
      ++p_issued;                                                                                \
      if (--p_left == 0 && p_issued < total) {                                                   \
        ++p_si;                                                                                  \
        const GemmSeg* sp = segs + p_si;                                                             \
        P_SETUP(sp->a_off, sp->b_off, sp->K, sp->a_sm, sp->a_sk, sp->b_sk, sp->b_sn)             \
      }                                                                                          \
    }                                                                                            \
    cp_commit();                                                                                 \
  }
#define CONSUME(SRC, AL, ALS)                                                                    \
  {                                                                                              \
    double ar[MT], ai[MT];                                                                       \
    cplx b[NT];                                                                                  \
    _Pragma("unroll") for (int i = 0; i < MT; ++i) {                                             \
      const cplx v = lds_c((SRC) + i * 512);                                                     \
      ar[i] = (AL) * v.x;                                                                        \
      ai[i] = (ALS) * v.y;                                                                       \
    }                                                                                            \
    _Pragma("unroll") for (int j = 0; j < NT; ++j) b[j] = lds_c((SRC) + (MT + j) * 512);         \
    _Pragma("unroll") for (int j = 0; j < NT; ++j)                                               \
      _Pragma("unroll") for (int i = 0; i < MT; ++i) dmma884(cre[i][j], ar[i], b[j].x);             \
    _Pragma("unroll") for (int j = 0; j < NT; ++j)                                               \
      _Pragma("unroll") for (int i = 0; i < MT; ++i) dmma884(cim[i][j], ar[i], b[j].y);             \
    _Pragma("unroll") for (int j = 0; j < NT; ++j)                                               \
      _Pragma("unroll") for (int i = 0; i < MT; ++i) dmma884(cre[i][j], -ai[i], b[j].y);            \
    _Pragma("unroll") for (int j = 0; j < NT; ++j)                                               \
      _Pragma("unroll") for (int i = 0; i < MT; ++i) dmma884(cim[i][j], ai[i], b[j].x);             \
  }

template <int MT, int NT>
__device__ __noinline__ void run_unit(const GemmUnit& u, const GemmSeg* __restrict__ segs, const cplx* __restrict__ A,
                                       const cplx* __restrict__ B, cplx* __restrict__ C, int lane, double conj_sign,
                                       uint32_t ring) {
  constexpr int D = RING_DEPTH;
  static_assert((D & (D - 1)) == 0, "RING_DEPTH must be a power of two");
  constexpr int F = MT + NT;
  constexpr int STAGE_BYTES = F * 512;
  double cre[MT][NT][2], cim[MT][NT][2];
#pragma unroll
  for (int i = 0; i < MT; ++i)
#pragma unroll
    for (int j = 0; j < NT; ++j) cre[i][j][0] = cre[i][j][1] = cim[i][j][0] = cim[i][j][1] = 0.0;
  const int total = u.steps;
  const int kq = lane & 3, r8 = lane >> 2;
  const uint32_t lane_ring = ring + lane * 16;
  if (total > 0) {
    int mi[MT], nj[NT];
#pragma unroll
    for (int i = 0; i < MT; ++i) mi[i] = min(u.m0 + 8 * i + r8, u.M - 1);
#pragma unroll
    for (int j = 0; j < NT; ++j) nj[j] = min(u.n0 + 8 * j + r8, u.N - 1);
    // ---- producer state
    const cplx* pa[MT];
    const cplx* pb[NT];
    int64_t dA, dB;
    int p_si = u.seg_begin, p_left, p_K, p_ask, p_bsk;  // p_left: steps left in the producer's segment
    const int se = u.seg_end;
    int p_issued = 0;
    P_SETUP(u.first.a_off, u.first.b_off, u.first.K, u.first.a_sm, u.first.a_sk, u.first.b_sk, u.first.b_sn)
#pragma unroll 1
    for (int d = 0; d < D - 1; ++d) { P_STEP_SLOW(lane_ring + d * STAGE_BYTES) }
    // ---- consumer state
    int c_si = u.seg_begin;
    int c_left = (u.first.K + 3) >> 2;
    double alpha = u.first.alpha;
    int t = 0;
    int n_cK = segs[min(c_si + 1, se - 1)].K;
    double n_alpha = segs[min(c_si + 1, se - 1)].alpha;
    while (t < total) {
      // chunk: steps during which the consumer stays in its segment and the producer issues only FULL
      // steps of its segment (p_left - 1 full steps are guaranteed when the last one may be ragged)
      const int p_full = (p_issued < total) ? ((p_K & 3) ? p_left - 1 : p_left) : 0;
      int n = min(c_left, p_full);
      const double als = alpha * conj_sign;
      if (n > 0) {
        c_left -= n;
        p_left -= n;
        p_issued += n;
#pragma unroll 1
        for (; n > 0; --n, ++t) {
          cp_wait<D - 2>();
          const uint32_t src = lane_ring + (t & (D - 1)) * STAGE_BYTES;
          const uint32_t dst = lane_ring + ((t + D - 1) & (D - 1)) * STAGE_BYTES;
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
          cp_commit();
          CONSUME(src, alpha, als)
        }
        if (p_left == 0 && p_issued < total) {
          ++p_si;
          const GemmSeg* sp = segs + p_si;
          P_SETUP(sp->a_off, sp->b_off, sp->K, sp->a_sm, sp->a_sk, sp->b_sk, sp->b_sn)
        }
      } else {
        // boundary step: slow producer path (ragged tail, segment switch or exhausted), one consumer step
        cp_wait<D - 2>();
        const uint32_t src = lane_ring + (t & (D - 1)) * STAGE_BYTES;
        P_STEP_SLOW(lane_ring + ((t + D - 1) & (D - 1)) * STAGE_BYTES)
        CONSUME(src, alpha, als)
        ++t;
        --c_left;
      }
      if (c_left == 0 && t < total) {
        ++c_si;
        c_left = (n_cK + 3) >> 2;
        alpha = n_alpha;
        n_cK = segs[min(c_si + 1, se - 1)].K;
        n_alpha = segs[min(c_si + 1, se - 1)].alpha;
      }
    }
    cp_wait<0>();
  }
  const int ec = kq * 2;
  cplx* gC = C + u.c_off;
#pragma unroll
  for (int i = 0; i < MT; ++i) {
    const int r = u.m0 + 8 * i + r8;
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
                                                           cplx* __restrict__ C, int conjA
) {
  __shared__ __align__(128) unsigned char ring_smem[RING_BYTES];
  const int lane = threadIdx.x;
  const int ui = blockIdx.x;
  if (ui >= nunits) return;
  pdl_launch_dependents();
  const GemmUnit u = units[ui];  // uploaded before the predecessor started: readable before the wait
  pdl_wait();
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

// Both stages of a two-stage contraction in one launch (UnitPair): block index = position in the joint unit list.
__global__ void __launch_bounds__(32) grouped_zgemm_pair_kernel(const GemmUnit* __restrict__ units, int nunits,
                                                                const GemmSeg* __restrict__ segs, const UnitLink* __restrict__ link,
                                                                const cplx* __restrict__ A1, const cplx* __restrict__ B1,
                                                                cplx* __restrict__ C1, const cplx* __restrict__ A2,
                                                                const cplx* __restrict__ B2, cplx* __restrict__ C2, int conj1,
                                                                int conj2, const int* __restrict__ dep_id,
                                                                const unsigned* __restrict__ dep_target,
                                                                unsigned* __restrict__ dep_cnt, unsigned epoch) {
  __shared__ __align__(128) unsigned char ring_smem[RING_BYTES];
  const int lane = threadIdx.x;
  const int ui = blockIdx.x;
  if (ui >= nunits) return;
  pdl_launch_dependents();
  const GemmUnit u = units[ui];
  const UnitLink lk = link[ui];
  pdl_wait();
  const uint32_t ring = (uint32_t)__cvta_generic_to_shared(ring_smem);
  const bool second = lk.stage != 0;
  if (second) {  // wait for the stage-1 outputs this unit reads (lanes share the list; every lane must see the data)
    for (int d = lk.dep_begin + lane; d < lk.dep_begin + lk.dep_count; d += 32) {
      const unsigned want = dep_target[d] * epoch;
      const unsigned* c = dep_cnt + dep_id[d];
      unsigned v;
      do {
        asm volatile("ld.acquire.gpu.u32 %0, [%1];" : "=r"(v) : "l"(c) : "memory");
      } while (v < want);
    }
    __syncwarp();
    __threadfence();
  }
  const cplx* A = second ? A2 : A1;
  const cplx* B = second ? B2 : B1;
  cplx* C = second ? C2 : C1;
  const double cs = (second ? conj2 : conj1) ? -1.0 : 1.0;
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
  if (!second) {  // this unit's part of its output is stored: publish it, then count
    __threadfence();
    __syncwarp();
    if (lane == 0) atomicAdd(dep_cnt + lk.sig, 1u);
  }
}

}  // namespace


void launch_grouped_gemm_pair(const UnitPair& pr, const cplx* A1, const cplx* B1, cplx* C1, const cplx* A2, const cplx* B2,
                              cplx* C2, unsigned* dep_counters, unsigned epoch, cudaStream_t s, int64_t* lc) {
  const int n = (int)pr.units.size();
  if (n == 0) return;
  launch_pdl(PDL_GEMM_FIRST, grouped_zgemm_pair_kernel, n, 32, s, (const GemmUnit*)pr.d_units, n, (const GemmSeg*)pr.d_segs,
             (const UnitLink*)pr.d_link, A1, B1, C1, A2, B2, C2, pr.conj1, pr.conj2, (const int*)pr.d_dep_id,
             (const unsigned*)pr.d_dep_target, dep_counters, epoch);
  ++*lc;
}

void launch_grouped_gemm(const Stage& st, const cplx* A, const cplx* B, cplx* C, cudaStream_t s, int64_t* lc,
                         int pdl_role) {
  const int n = (int)st.units.size();
  if (n == 0) return;
  launch_pdl(pdl_role, grouped_zgemm_kernel, n, 32, s, (const GemmUnit*)st.d_units, n, (const GemmSeg*)st.d_segs, A, B, C,
             st.opA != OPA_N ? 1 : 0);
  ++*lc;
}

}  // namespace fh
