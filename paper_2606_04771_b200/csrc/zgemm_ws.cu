// Warp-specialised persistent form of the segmented grouped complex128 GEMM:
//     C_o (M x N) = sum_{t in seg(o)} alpha_t * op(A_t) (M x K_t) * op(B_t) (K_t x N),  alpha_t real,
// and of TWO such stages that feed one another (H1 -> H2: Z = L theta, H theta = Z R^T) in ONE launch.
//
// Why a second form.  With one warp-unit per one-warp CTA (zgemm.cu) every unit pays its own start-up latency
// (descriptor, first operand fragments, epilogue, CTA turnover) and every warp issues its own copies.  Here the
// memory side is taken off the warps that issue DMMAs (DESIGN.md 6.2 has the measurements that say where each
// form wins; the library picks per plan):
//   * one persistent CTA per SM, 12 warps: 8 consumers (two per sub-partition) in two independent groups of
//     four, and a producer warp group (two producer warps per consumer group).  After the barriers are set up
//     the producers drop to 88 registers and the consumers rise to 208 (setmaxnreg; 8 x 208 + 4 x 88 = 12 x 168,
//     the register pool the CTA is launched with);
//   * a consumer group works on one TILE: up to 64 x 64 of an output block over (a k range of) its concatenated
//     segments.  Its four warps share the tile in the arrangement the host found best for the tile's shape:
//     2 x 2 quadrants (parts up to 4 x 4 sub-tiles of 8 x 8), four column strips or four row strips (parts up
//     to 8 x 2 / 2 x 8); the second group takes the parts in mirrored order so that the two warps of a
//     sub-partition hold opposite parts;
//   * the producers of a group walk the tile queue (heaviest first, one atomic ticket counter; the leader takes
//     the tickets and passes them to the follower through a mailbox in shared memory) and stream the operand
//     panels of their group -- the leader the A panels, the follower the B panels, 16 k at a time, cp.async
//     (LDGSTS) with zero fill beyond a segment's K -- into the group's 3-stage ring; a stage is handed over by
//     an mbarrier that counts the cp.async completions of both producers (cp.async.mbarrier.arrive.noinc) and
//     the write of the 64-byte stage descriptor (alpha, k-steps, first / last flags, tile geometry), and is
//     handed back by the four consumer warps through a second mbarrier.  The ring runs on across tile
//     boundaries: between two tiles the consumers only store their accumulators;
//   * consumers execute LDS.128 from XOR-swizzled panels (conflict free for either operand orientation), the
//     two DMULs that fold alpha into an A fragment, and DMMA.8x8x4 (four real DMMAs per complex product);
//   * two stages in one launch: the queue holds the stage-1 tiles, then the stage-2 tiles.  Every warp that
//     has stored its part of a stage-1 output panel raises that panel's counter (fence + atomic); a producer
//     starts a stage-2 tile only when the panels the tile reads have all their arrivals (ld.acquire).  Tickets
//     are handed out in queue order, so everything a waiting producer waits for is already being worked on;
//   * a tile heavier than the even share of a group is split along k: the later parts leave their accumulators
//     in scratch, the part that starts at k = 0 adds them in slot order (fixed order: deterministic) and stores.
// Outputs are never shared between warps, the k order inside a part is the task-list order, parts are added in
// a fixed order: results are bit-identical from run to run.
#include "fh_internal.hpp"

namespace fh {

namespace {

constexpr int WS_GROUPS = 2;
constexpr int WS_STAGES = 3;
constexpr int WS_PANEL = 64 * 16 * 16;         // one operand panel of a stage: 64 rows x 16 k x 16 B
constexpr int WS_STAGE_BYTES = 2 * WS_PANEL;   // A panel + B panel
constexpr int WS_META = 64;
constexpr int WS_NCONS = 8;                    // consumer warps
constexpr int WS_THREADS = 32 * (WS_NCONS + 4);  // two consumer warp groups + one producer warp group
constexpr int WS_DATA_BYTES = WS_GROUPS * WS_STAGES * WS_STAGE_BYTES;
constexpr int WS_SMEM_BYTES = WS_DATA_BYTES + WS_GROUPS * WS_STAGES * (WS_META + 16) + WS_GROUPS * 32;

enum { F_FIRST = 1, F_LAST = 2, F_EXIT = 4 };

// operand sets of the (up to) two stages of a launch, and the cross-stage dependency tables
struct WsArgs {
  const cplx* A[2];
  const cplx* B[2];
  cplx* C[2];
  int conj[2];
  const int* dep_id;
  const unsigned* dep_target;
  unsigned* dep_cnt;   // nullptr: single stage, nothing to signal
  unsigned epoch;
};

__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c[0]), "+d"(c[1])
               : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(uint32_t smem_addr, const void* gptr, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_addr), "l"(gptr), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ cplx lds_c(uint32_t addr) {
  cplx v;
  asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  return v;
}
__device__ __forceinline__ int4 lds_i4(uint32_t addr) {
  int4 v;
  asm volatile("ld.shared.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts_i4(uint32_t addr, int4 v) {
  asm volatile("st.shared.v4.s32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void mbar_init(uint32_t a, int count) {
  asm volatile("mbarrier.init.shared.b64 [%0], %1;" ::"r"(a), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t a) {
  asm volatile("mbarrier.arrive.shared.b64 _, [%0];" ::"r"(a) : "memory");
}
// arrives (without raising the expected count) once all cp.async of this thread issued so far have landed
__device__ __forceinline__ void mbar_arrive_cp(uint32_t a) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared.b64 [%0];" ::"r"(a) : "memory");
}
__device__ __forceinline__ bool mbar_try(uint32_t a, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(a), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t a, uint32_t parity) {
  while (!mbar_try(a, parity)) {
  }
}


struct SmemMap {
  uint32_t data, meta, full, empty, mail;  // shared-space addresses of the regions
  __device__ __forceinline__ uint32_t stage(int g, int s) const { return data + (g * WS_STAGES + s) * WS_STAGE_BYTES; }
  __device__ __forceinline__ uint32_t meta_of(int g, int s) const { return meta + (g * WS_STAGES + s) * WS_META; }
  __device__ __forceinline__ uint32_t full_of(int g, int s) const { return full + (g * WS_STAGES + s) * 8; }
  __device__ __forceinline__ uint32_t empty_of(int g, int s) const { return empty + (g * WS_STAGES + s) * 8; }
};

// ------------------------------------------------------------------------------------------------ consumer
// Panel layouts (16-byte elements e):
//   K-contiguous operand (a_sk == 1 / b_sk == 1): panel[row][k], row pitch 256 B, element (row, k) at
//       row * 256 + ((k ^ 4 (row & 1)) * 16)        -- rows r, r+1 of a quarter warp fall into different 64-byte halves
//   row-contiguous operand (a_sm == 1 / b_sn == 1): panel[k][row], k pitch 1024 B, element (k, row) at
//       k * 1024 + ((row ^ 2 (k & 3)) * 16)          -- the four k of a quarter warp fall into different 32-byte slots
// DMMA.8x8x4 fragments: lane l holds A[row l / 4][k l % 4] and B[k l % 4][col l / 4].
struct LaneAddr {
  uint32_t base;     // lane part of the address inside a panel (sub-tile 0, k-step 0)
  uint32_t istride;  // bytes from sub-tile i to i + 1
  uint32_t rc;       // 1: row-contiguous layout
};
__device__ __forceinline__ LaneAddr lane_addr(int rc, int sub0, int r8, int kq) {
  LaneAddr a;
  a.rc = rc;
  if (rc) {
    a.base = kq * 1024 + (8 * sub0 + (r8 ^ (2 * kq))) * 16;
    a.istride = 128;
  } else {
    a.base = (8 * sub0 + r8) * 256 + kq * 16;
    a.istride = 2048;
  }
  return a;
}
__device__ __forceinline__ uint32_t step_off(const LaneAddr& a, int s, int r8) {
  return a.rc ? (uint32_t)s * 4096u : (uint32_t)((s ^ (r8 & 1)) << 6);
}

struct ChunkHead {
  int flags, nsteps;
  double alpha;
};
__device__ __forceinline__ ChunkHead read_head(uint32_t meta) {
  const int4 v = lds_i4(meta);
  ChunkHead h;
  h.flags = v.x;
  h.nsteps = v.y;
  h.alpha = __hiloint2double(v.w, v.z);
  return h;
}

// ring position of a consumer: stage | phase << 8
// One body per register-tile shape MTM x NTM (sub-tiles of 8 x 8; MTM * NTM <= 16): shapes up to 4 x 4 for the
// quadrant arrangement, up to 8 x 2 / 2 x 8 for the strip arrangements.
template <int MTM, int NTM>
__device__ __forceinline__ int consume_tile(const SmemMap sm, int g, int pos, ChunkHead hd, int sub_m0, int sub_n0,
                                         int quad, const WsArgs& ar, int lane, cplx* __restrict__ scratch,
                                         unsigned* __restrict__ pflags, unsigned ptarget) {
  constexpr int mt = MTM, nt = NTM;
  int stage = pos & 0xff;
  uint32_t phase = (uint32_t)pos >> 8;
  const int kq = lane & 3, r8 = lane >> 2;
  // tile geometry (first chunk's descriptor)
  const uint32_t m0a = sm.meta_of(g, stage);
  const int4 g1 = lds_i4(m0a + 16), g2 = lds_i4(m0a + 32), g3 = lds_i4(m0a + 48);
  const int64_t c_off = ((int64_t)(uint32_t)g1.y << 32) | (uint32_t)g1.x;
  const int ldc = g1.z, M = g1.w, N = g2.x, tm0 = g2.y, tn0 = g2.z;
  const LaneAddr la = lane_addr(g3.x & 1, sub_m0, r8, kq), lb = lane_addr((g3.x >> 1) & 1, sub_n0, r8, kq);
  const int slot = g3.y, kind = g3.w & 3, nparts = (g3.w >> 4) & 255, tstage = (g3.x >> 2) & 1, sig = (g3.x >> 3) - 1;
  cplx* __restrict__ C = tstage ? ar.C[1] : ar.C[0];
  const double conj_sign = (tstage ? ar.conj[1] : ar.conj[0]) ? -1.0 : 1.0;
  double cre[MTM][NTM][2], cim[MTM][NTM][2];
#pragma unroll
  for (int i = 0; i < MTM; ++i)
#pragma unroll
    for (int j = 0; j < NTM; ++j) cre[i][j][0] = cre[i][j][1] = cim[i][j][0] = cim[i][j][1] = 0.0;
  for (;;) {
    const uint32_t sa = sm.stage(g, stage) + la.base, sb = sm.stage(g, stage) + WS_PANEL + lb.base;
    const double al = hd.alpha, als = hd.alpha * conj_sign;
#pragma unroll 1
    for (int s = 0; s < hd.nsteps; ++s) {
      const uint32_t pa = sa + step_off(la, s, r8), pb = sb + step_off(lb, s, r8);
      // the operand with the fewer fragments stays in registers for the whole k-step, the other is read just
      // before its DMMAs; consecutive DMMAs never hit the same accumulator
      if (MTM <= NTM) {
        double ar_[MTM], ai_[MTM];
#pragma unroll
        for (int i = 0; i < MTM; ++i)
          if (i < mt) {
            const cplx v = lds_c(pa + i * la.istride);
            ar_[i] = al * v.x;
            ai_[i] = als * v.y;
          }
#pragma unroll
        for (int j = 0; j < NTM; ++j)
          if (j < nt) {
            const cplx b = lds_c(pb + j * lb.istride);
#pragma unroll
            for (int i = 0; i < MTM; ++i)
              if (i < mt) dmma884(cre[i][j], ar_[i], b.x);
#pragma unroll
            for (int i = 0; i < MTM; ++i)
              if (i < mt) dmma884(cim[i][j], ar_[i], b.y);
#pragma unroll
            for (int i = 0; i < MTM; ++i)
              if (i < mt) dmma884(cre[i][j], -ai_[i], b.y);
#pragma unroll
            for (int i = 0; i < MTM; ++i)
              if (i < mt) dmma884(cim[i][j], ai_[i], b.x);
          }
      } else {
        cplx b[NTM];
#pragma unroll
        for (int j = 0; j < NTM; ++j)
          if (j < nt) b[j] = lds_c(pb + j * lb.istride);
#pragma unroll
        for (int i = 0; i < MTM; ++i)
          if (i < mt) {
            const cplx v = lds_c(pa + i * la.istride);
            const double ar_ = al * v.x, ai_ = als * v.y;
#pragma unroll
            for (int j = 0; j < NTM; ++j)
              if (j < nt) dmma884(cre[i][j], ar_, b[j].x);
#pragma unroll
            for (int j = 0; j < NTM; ++j)
              if (j < nt) dmma884(cim[i][j], ar_, b[j].y);
#pragma unroll
            for (int j = 0; j < NTM; ++j)
              if (j < nt) dmma884(cre[i][j], -ai_, b[j].y);
#pragma unroll
            for (int j = 0; j < NTM; ++j)
              if (j < nt) dmma884(cim[i][j], ai_, b[j].x);
          }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(sm.empty_of(g, stage));
    const int last = hd.flags & F_LAST;
    if (++stage == WS_STAGES) {
      stage = 0;
      phase ^= 1;
    }
    if (last) break;
    mbar_wait(sm.full_of(g, stage), phase);
    hd = read_head(sm.meta_of(g, stage));
  }
  // k-split tiles: accumulators travel through scratch in fragment order (lane-contiguous: coalesced)
  if (kind == 1) {
    cplx* sp = scratch + (size_t)slot * WS_SLOT_ELEMS + (size_t)quad * 1024 + lane;
#pragma unroll
    for (int i = 0; i < MTM; ++i)
#pragma unroll
      for (int j = 0; j < NTM; ++j)
        if (i < mt && j < nt) {
          sp[((i * NTM + j) * 2 + 0) * 32] = make_double2(cre[i][j][0], cim[i][j][0]);
          sp[((i * NTM + j) * 2 + 1) * 32] = make_double2(cre[i][j][1], cim[i][j][1]);
        }
    __threadfence();
    __syncwarp();
    if (lane == 0) atomicAdd(pflags + slot, 1u);
    return stage | (int)(phase << 8);
  }
  for (int p = 0; p < nparts; ++p) {
    if (lane == 0) {
      const volatile unsigned* f = pflags + slot + p;
      while (*f < ptarget) {
      }
    }
    __syncwarp();
    __threadfence();
    const cplx* sp = scratch + (size_t)(slot + p) * WS_SLOT_ELEMS + (size_t)quad * 1024 + lane;
#pragma unroll
    for (int i = 0; i < MTM; ++i)
#pragma unroll
      for (int j = 0; j < NTM; ++j)
        if (i < mt && j < nt) {
          const cplx v0 = __ldcg(sp + ((i * NTM + j) * 2 + 0) * 32), v1 = __ldcg(sp + ((i * NTM + j) * 2 + 1) * 32);
          cre[i][j][0] += v0.x;
          cim[i][j][0] += v0.y;
          cre[i][j][1] += v1.x;
          cim[i][j][1] += v1.y;
        }
  }
  const int ec = kq * 2;
  cplx* gC = C + c_off;
#pragma unroll
  for (int i = 0; i < MTM; ++i) {
    const int r = tm0 + 8 * (sub_m0 + i) + r8;
    if (i < mt && r < M) {
#pragma unroll
      for (int j = 0; j < NTM; ++j) {
        const int c = tn0 + 8 * (sub_n0 + j) + ec;
        cplx* p = gC + (int64_t)r * ldc + c;
        if (j < nt && c < N) p[0] = make_double2(cre[i][j][0], cim[i][j][0]);
        if (j < nt && c + 1 < N) p[1] = make_double2(cre[i][j][1], cim[i][j][1]);
      }
    }
  }
  if (ar.dep_cnt && sig >= 0) {  // this warp's part of the output panel is in memory: let its readers know
    __threadfence();
    __syncwarp();
    if (lane == 0) atomicAdd(ar.dep_cnt + sig, 1u);
  }
  return stage | (int)(phase << 8);
}

// a warp whose part of the tile is empty still takes part in the stage hand-over
__device__ __forceinline__ int skip_tile(const SmemMap sm, int g, int pos, ChunkHead hd, int lane,
                                      unsigned* __restrict__ pflags, unsigned* __restrict__ dep_cnt) {
  int stage = pos & 0xff;
  uint32_t phase = (uint32_t)pos >> 8;
  {  // an empty part still counts towards the four arrivals of a k-split slot / of an output panel
    const int4 g3 = lds_i4(sm.meta_of(g, stage) + 48);
    if (lane == 0) {
      if ((g3.w & 3) == 1) atomicAdd(pflags + g3.y, 1u);
      else if (dep_cnt && (g3.x >> 3) > 0) atomicAdd(dep_cnt + (g3.x >> 3) - 1, 1u);
    }
  }
  for (;;) {
    __syncwarp();
    if (lane == 0) mbar_arrive(sm.empty_of(g, stage));
    const int last = hd.flags & F_LAST;
    if (++stage == WS_STAGES) {
      stage = 0;
      phase ^= 1;
    }
    if (last) break;
    mbar_wait(sm.full_of(g, stage), phase);
    hd = read_head(sm.meta_of(g, stage));
  }
  return stage | (int)(phase << 8);
}

// part q (0..3) of `n` sub-tiles cut into `parts` nearly equal consecutive ranges
__device__ __forceinline__ void split_range(int n, int parts, int q, int& begin, int& count) {
  const int base = n / parts, extra = n % parts;
  begin = q * base + min(q, extra);
  count = base + (q < extra ? 1 : 0);
}

__device__ __forceinline__ void consumer_loop(const SmemMap sm, int g, int wq, const WsArgs& ar, int lane,
                                              cplx* __restrict__ scratch, unsigned* __restrict__ pflags, unsigned ptarget) {
  // The four warps of a group share a tile in one of three arrangements chosen per tile by the host (the one
  // whose largest part is smallest): 2 x 2 quadrants, four column strips, four row strips.  The second group
  // takes the parts in mirrored order, so that the two warps that share a sub-partition hold opposite parts
  // (a tile's larger parts are its first ones).
  const int q = g == 0 ? wq : 3 - wq;
  int pos = 0;
  for (;;) {
    const int stage = pos & 0xff;
    mbar_wait(sm.full_of(g, stage), (uint32_t)pos >> 8);
    const uint32_t ma = sm.meta_of(g, stage);
    const ChunkHead hd = read_head(ma);
    if (hd.flags & F_EXIT) {
      break;
    }
    const int h = lds_i4(ma + 32).w;
    const int4 g3 = lds_i4(ma + 48);
    const int w = g3.z, arr = (g3.w >> 2) & 3;
    int sm0, mt, sn0, nt;
    if (arr == 0) {
      split_range(h, 2, q >> 1, sm0, mt);
      split_range(w, 2, q & 1, sn0, nt);
    } else if (arr == 1) {
      sm0 = 0;
      mt = h;
      split_range(w, 4, q, sn0, nt);
    } else {
      split_range(h, 4, q, sm0, mt);
      sn0 = 0;
      nt = w;
    }
    if (mt == 0 || nt == 0) {
      pos = skip_tile(sm, g, pos, hd, lane, pflags, ar.dep_cnt);
      continue;
    }
    switch (mt * 16 + nt) {
#define WS_CASE(MT, NT)                                                                                             \
  case MT * 16 + NT:                                                                                                \
    pos = consume_tile<MT, NT>(sm, g, pos, hd, sm0, sn0, q, ar, lane, scratch, pflags, ptarget);              \
    break;
      WS_CASE(1, 1) WS_CASE(1, 2) WS_CASE(1, 3) WS_CASE(1, 4) WS_CASE(2, 1) WS_CASE(2, 2) WS_CASE(2, 3) WS_CASE(2, 4)
      WS_CASE(3, 1) WS_CASE(3, 2) WS_CASE(3, 3) WS_CASE(3, 4) WS_CASE(4, 1) WS_CASE(4, 2) WS_CASE(4, 3) WS_CASE(4, 4)
      WS_CASE(5, 1) WS_CASE(5, 2) WS_CASE(6, 1) WS_CASE(6, 2) WS_CASE(7, 1) WS_CASE(7, 2) WS_CASE(8, 1) WS_CASE(8, 2)
      WS_CASE(1, 5) WS_CASE(2, 5) WS_CASE(1, 6) WS_CASE(2, 6) WS_CASE(1, 7) WS_CASE(2, 7) WS_CASE(1, 8) WS_CASE(2, 8)
#undef WS_CASE
      default:
        pos = skip_tile(sm, g, pos, hd, lane, pflags, ar.dep_cnt);
        break;
    }
  }
}

// ------------------------------------------------------------------------------------------------ producer
// Two producer warps per consumer group walk the same tile sequence: the LEADER copies the A panels, takes the
// tickets of the tile queue and writes the stage descriptors; the FOLLOWER copies the B panels and learns each
// ticket from a four-entry mailbox in shared memory (the leader is never more than WS_STAGES <= 3 chunks, hence
// tiles, ahead: a stage is handed to the consumers only when both producers have filled their half).
struct ProdState {
  WsTile t;     // current tile (t.first = its first segment)
  GemmSeg s;    // current segment
  GemmSeg nx;   // the segment after it (loaded when s became current)
  int seg, k0, valid, stage, first, seq, rem, ticket, have_ticket;
  uint32_t phase;
};

// The leader takes the ticket of the NEXT tile when three chunks of the current one remain (result left pending:
// no round trip on the critical path), late enough that a group does not sit on a heavy tile it will not start
// for a long time -- heaviest-first order is what balances a launch of a few tiles per group.
__device__ __forceinline__ void take_ticket(ProdState& st, unsigned* counter, int lane) {
  if (lane == 0) st.ticket = (int)atomicAdd(counter, 1u);
  st.have_ticket = 1;
}

// next tile of the queue: the ticket (leader: one atomic; follower: the mailbox), then ONE 128-byte load that
// also carries the tile's first segment
__device__ __forceinline__ void load_tile(ProdState& st, int role, uint32_t mailbox, const WsTile* __restrict__ tiles,
                                          int ntiles, const GemmSeg* __restrict__ segs, unsigned* counter, int lane,
                                          const WsArgs& ar) {
  const uint32_t slot = mailbox + (st.seq & 3) * 8;
  int idx = 0;
  if (role == 0) {
    if (!st.have_ticket) take_ticket(st, counter, lane);
    st.have_ticket = 0;
    if (lane == 0) {
      idx = st.ticket;
      asm volatile("st.volatile.shared.v2.u32 [%0], {%1, %2};" ::"r"(slot), "r"(idx), "r"(st.seq + 1) : "memory");
    }
  } else if (lane == 0) {
    int stamp;
    do {
      asm volatile("ld.volatile.shared.v2.u32 {%0, %1}, [%2];" : "=r"(idx), "=r"(stamp) : "r"(slot) : "memory");
    } while (stamp != st.seq + 1);
  }
  ++st.seq;
  idx = __shfl_sync(0xffffffffu, idx, 0);
  st.valid = idx < ntiles;
  if (!st.valid) return;
  st.t = tiles[idx];  // every lane reads the same 128 bytes: broadcast transactions
  st.s = st.t.first;
  st.seg = st.t.seg_begin;
  st.k0 = st.t.k_begin;
  st.first = 1;
  st.rem = st.t.nparts >> 8;  // chunks of the tile not yet issued
  if (st.seg + 1 < st.t.seg_end) st.nx = segs[st.seg + 1];
  // a tile of the second stage waits until the first-stage panels it reads are complete
  if (st.t.dep_count > 0 && ar.dep_cnt) {
    for (int d = lane; d < st.t.dep_count; d += 32) {
      const unsigned* c = ar.dep_cnt + ar.dep_id[st.t.dep_begin + d];
      const unsigned target = ar.dep_target[st.t.dep_begin + d] * ar.epoch;
      unsigned v;
      do {
        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(c) : "memory");
      } while (v < target);
    }
    __syncwarp();
  }
}

// copies one operand panel of the chunk [k0, k0 + nk) of the current segment into a stage.
//   nrow: valid rows of the panel (rows of the tile inside the block; the panel rows beyond are never stored, so
//   they are left as they are); r0: first row of the tile inside the block; k >= K is zero-filled (a zero-size
//   cp.async reads nothing, whatever its source address).
__device__ __forceinline__ void copy_panel(uint32_t dst, const cplx* __restrict__ base, int64_t s_row, int64_t s_k,
                                           int nrow, int r0, int k0, int K, int nk, int lane) {
  if (s_k == 1) {  // K-contiguous: panel[row][k]; a half warp copies the 16 k of one row, a warp two rows
    const int kk = lane & 15, rl = lane >> 4;
    if (kk >= nk) return;
    const int sz = (k0 + kk < K) ? 16 : 0;
    const cplx* p = base + (int64_t)(r0 + rl) * s_row + (k0 + kk);
    const int64_t step = 2 * s_row;
    uint32_t d = dst + rl * 256 + ((kk ^ (4 * rl)) * 16);
    const int n = nrow - rl;  // this lane copies rows rl, rl + 2, ... < nrow
#pragma unroll 4
    for (int it = 0; it < n; it += 2) {
      cp_async16(d, p, sz);
      p += step;
      d += 512;
    }
  } else {  // row-contiguous: panel[k][row]; a warp copies 32 rows of one k
    const cplx* p = base + (int64_t)k0 * s_k + (int64_t)(r0 + lane) * s_row;
    const bool v0 = lane < nrow, v1 = lane + 32 < nrow;
    const uint32_t d0 = dst + lane * 16;
#pragma unroll 4
    for (int kk = 0; kk < nk; ++kk) {
      const int sz = (k0 + kk < K) ? 16 : 0;
      const uint32_t x = (uint32_t)(2 * (kk & 3)) * 16;
      if (v0) cp_async16((d0 ^ x) + kk * 1024, p, sz);
      if (v1) cp_async16(((d0 + 512) ^ x) + kk * 1024, p + 32 * s_row, sz);
      p += s_k;
    }
  }
}

__device__ __forceinline__ void producer_loop(const SmemMap sm, int g, int role, const WsTile* __restrict__ tiles,
                                              int ntiles, const GemmSeg* __restrict__ segs, const WsArgs& ar,
                                              unsigned* counters, int lane) {
  ProdState st;
  st.stage = 0;
  st.phase = 0;
  st.seq = 0;
  st.ticket = 0;
  st.have_ticket = 0;
  const uint32_t mailbox = sm.mail + g * 32;
  load_tile(st, role, mailbox, tiles, ntiles, segs, counters, lane, ar);
  for (;;) {
    mbar_wait(sm.empty_of(g, st.stage), st.phase ^ 1);
    const uint32_t full = sm.full_of(g, st.stage), meta = sm.meta_of(g, st.stage);
    if (!st.valid) {
      if (role == 0 && lane == 0) {
        sts_i4(meta, make_int4(F_EXIT | F_LAST, 0, 0, 0));
        mbar_arrive(full);
      }
      mbar_arrive_cp(full);
      break;
    }
    int flags = st.first ? F_FIRST : 0, nsteps = 0;
    double alpha = 0.0;
    const bool has_seg = st.seg < st.t.seg_end;
    const int a_rc = has_seg ? (st.s.a_sk == 1 ? 0 : 1) : 0, b_rc = has_seg ? (st.s.b_sk == 1 ? 0 : 1) : 0;
    if (has_seg) {
      const int K = (st.seg == st.t.seg_end - 1) ? min(st.s.K, st.t.k_end) : st.s.K;  // a k-split part may end early
      int nk = min(16, K - st.k0);
      nk = (nk + 3) & ~3;  // whole DMMA k-steps; k >= K is zero-filled
      nsteps = nk >> 2;
      alpha = st.s.alpha;
      const uint32_t da = sm.stage(g, st.stage);
      const cplx* __restrict__ A = (st.t.stage_sig & 1) ? ar.A[1] : ar.A[0];
      const cplx* __restrict__ B = (st.t.stage_sig & 1) ? ar.B[1] : ar.B[0];
      {
        if (role == 0)
          copy_panel(da, A + st.s.a_off, st.s.a_sm, st.s.a_sk, min(8 * st.t.h, st.t.M - st.t.m0), st.t.m0, st.k0, K, nk, lane);
        else
          copy_panel(da + WS_PANEL, B + st.s.b_off, st.s.b_sn, st.s.b_sk, min(8 * st.t.w, st.t.N - st.t.n0), st.t.n0, st.k0, K, nk, lane);
      }
      st.k0 += 16;
      if (st.k0 >= K) {
        ++st.seg;
        st.k0 = 0;
      }
    }
    const bool last = !(st.seg < st.t.seg_end);
    if (--st.rem == 3 && role == 0) take_ticket(st, counters, lane);
    if (role == 0 && lane == 0) {
      if (last) flags |= F_LAST;
      sts_i4(meta, make_int4(flags, nsteps, __double2loint(alpha), __double2hiint(alpha)));
      if (st.first) {
        sts_i4(meta + 16, make_int4((int)(uint32_t)(st.t.c_off & 0xffffffffll), (int)(st.t.c_off >> 32), st.t.ldc, st.t.M));
        sts_i4(meta + 32, make_int4(st.t.N, st.t.m0, st.t.n0, st.t.h));
        sts_i4(meta + 48, make_int4(a_rc | (b_rc << 1) | ((st.t.stage_sig & 1) << 2) | ((st.t.stage_sig >> 1) << 3), st.t.slot,
                                    st.t.w, st.t.kind | ((st.t.nparts & 255) << 4)));  // kind = part kind | arrangement << 2
      }
      mbar_arrive(full);
    }
    st.first = 0;
    mbar_arrive_cp(full);
    if (++st.stage == WS_STAGES) {
      st.stage = 0;
      st.phase ^= 1;
    }
    if (last) {
      load_tile(st, role, mailbox, tiles, ntiles, segs, counters, lane, ar);
    } else if (st.k0 == 0) {  // segment switch: the next one was requested when this one started
      st.s = st.nx;
      if (st.seg + 1 < st.t.seg_end) st.nx = segs[st.seg + 1];
    }
  }
}

__global__ void __launch_bounds__(WS_THREADS, 1)
    grouped_zgemm_ws_kernel(const WsTile* __restrict__ tiles, int ntiles, const GemmSeg* __restrict__ segs,
                            const WsArgs ar, unsigned* __restrict__ counters, cplx* __restrict__ scratch,
                            unsigned* __restrict__ pflags, unsigned ptarget) {
  extern __shared__ __align__(1024) unsigned char ws_smem[];
  SmemMap sm;
  sm.data = (uint32_t)__cvta_generic_to_shared(ws_smem);
  sm.meta = sm.data + WS_DATA_BYTES;
  sm.full = sm.meta + WS_GROUPS * WS_STAGES * WS_META;
  sm.empty = sm.full + WS_GROUPS * WS_STAGES * 8;
  sm.mail = sm.empty + WS_GROUPS * WS_STAGES * 8;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int i = 0; i < WS_GROUPS * WS_STAGES; ++i) {
      mbar_init(sm.full + 8 * i, 65);   // 2 x 32 cp.async arrivals of the two producer warps + the descriptor write
      mbar_init(sm.empty + 8 * i, 4);   // the four consumer warps of the group
    }
    for (int i = 0; i < WS_GROUPS * 8; ++i)
      asm volatile("st.shared.u32 [%0], %1;" ::"r"(sm.mail + 4 * i), "r"(0) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (warp >= WS_NCONS) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 88;");
    const int g = (warp - WS_NCONS) & 1, role = (warp - WS_NCONS) >> 1;
    producer_loop(sm, g, role, tiles, ntiles, segs, ar, counters, lane);
    // the leader that finishes last (over all CTAs) re-arms the queue for the next launch
    if (role == 0 && lane == 0) {
      __threadfence();
      const unsigned n = gridDim.x * WS_GROUPS;
      if (atomicInc(counters + 1, n - 1) == n - 1) atomicExch(counters, 0u);
    }
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 208;");
    consumer_loop(sm, warp >> 2, warp & 3, ar, lane, scratch, pflags, ptarget);
  }
}

}  // namespace

int ws_smem_bytes() { return WS_SMEM_BYTES; }

static void ws_launch(const WsTile* d_tiles, int n, const GemmSeg* d_segs, const WsArgs& ar, unsigned* d_counters, int grid,
                      cplx* scratch, unsigned* flags, cudaStream_t s) {
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(grouped_zgemm_ws_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, WS_SMEM_BYTES);
    attr_set = true;
  }
  const int g = grid < 1 ? 1 : grid;
  grouped_zgemm_ws_kernel<<<g, WS_THREADS, WS_SMEM_BYTES, s>>>(d_tiles, n, d_segs, ar, d_counters, scratch, flags,
                                                            4u * ar.epoch);
}

void launch_grouped_gemm_ws(const Stage& st, const cplx* A, const cplx* B, cplx* C, unsigned* d_counters, int grid,
                            cplx* scratch, unsigned* flags, unsigned epoch, cudaStream_t s, int64_t* lc) {
  const int n = (int)st.tiles.size();
  if (n == 0) return;
  WsArgs ar = {};
  ar.A[0] = A;
  ar.B[0] = B;
  ar.C[0] = C;
  ar.conj[0] = st.opA != OPA_N ? 1 : 0;
  ar.epoch = epoch;
  ws_launch(st.d_tiles, n, st.d_segs, ar, d_counters, grid, scratch, flags, s);
  ++*lc;
}

void launch_grouped_gemm_ws_pair(const WsPair& pr, const cplx* A1, const cplx* B1, cplx* C1, const cplx* A2, const cplx* B2,
                                 cplx* C2, unsigned* d_counters, int grid, cplx* scratch, unsigned* flags,
                                 unsigned* dep_counters, unsigned epoch, cudaStream_t s, int64_t* lc) {
  const int n = (int)pr.tiles.size();
  if (n == 0) return;
  WsArgs ar = {};
  ar.A[0] = A1;
  ar.B[0] = B1;
  ar.C[0] = C1;
  ar.A[1] = A2;
  ar.B[1] = B2;
  ar.C[1] = C2;
  ar.conj[0] = pr.conj1;
  ar.conj[1] = pr.conj2;
  ar.dep_id = pr.d_dep_id;
  ar.dep_target = pr.d_dep_target;
  ar.dep_cnt = dep_counters;
  ar.epoch = epoch;
  ws_launch(pr.d_tiles, n, pr.d_segs, ar, d_counters, grid, scratch, flags, s);
  ++*lc;
}

}  // namespace fh
