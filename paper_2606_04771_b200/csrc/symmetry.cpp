// Host symmetry layer: labels, fusion rules, reduced MPO, task lists.
//
// Canonical orders (must match what DESIGN.md states; the oracle emits the same lists from its
// own code and the tests compare the integer tuples bit for bit):
//   * blocks of a tensor: lexicographic in the flattened label tuple, sectors ordered by (q, tj);
//   * stage-1 tasks of a left contraction: by output key (a',s',c',w', rest of the ket key),
//     segments by (w, a, s);
//   * two-site stage 2: by output key, segments by (c, s2, b, w_m, w_r);
//   * one-site stage 2: by output key, segments by (c, w');
//   * left-environment stage 2: by output key (c',w',c), segments by (a', s');
//   * right-environment stage 2: by output key (c',w,c), segments by (s', b', w', s, b).
#include "symmetry.hpp"

#include <algorithm>
#include <cmath>
#include <stdexcept>

namespace fh {

// ----------------------------------------------------------------------------- symmetry modes
const SymMode SYM_SU2 = {0, 3, 4, {1, -1, 0, 0}, {0, 0, 1, 0}, {0, 1, -1, 0, 0, 0}, {0, 1, 1, 0, 0, 0}};
const SymMode SYM_U1U1 = {1, 4, 6, {-64, 1, -1, 64}, {0, 0, 0, 0}, {0, 65, 63, -65, -63, 0}, {0, 0, 0, 0, 0, 0}};
static thread_local const SymMode* t_sym = &SYM_SU2;
const SymMode& sym() { return *t_sym; }
SymScope::SymScope(const SymMode* m) : prev(t_sym) { t_sym = m ? m : &SYM_SU2; }
SymScope::~SymScope() { t_sym = prev; }

// ----------------------------------------------------------------------------- Bond / BlockTensor
int Bond::find(Sector s) const {
  auto it = std::lower_bound(sec.begin(), sec.end(), s);
  if (it == sec.end() || !(*it == s)) return -1;
  return (int)(it - sec.begin());
}
int Bond::chi_full() const {  // Eq. (8)
  int x = 0;
  for (size_t i = 0; i < sec.size(); ++i) x += d[i] * (sec[i].tj + 1);
  return x;
}
int Bond::chi_su2() const {  // Eq. (10)
  int x = 0;
  for (int v : d) x += v;
  return x;
}
int Bond::dmax() const {  // Eq. (9)
  int x = 0;
  for (int v : d) x = std::max(x, v);
  return x;
}

void BlockTensor::clear() {
  keys.clear();
  rows.clear();
  cols.clear();
  off.clear();
  ld.clear();
  col0.clear();
  index.clear();
  nelem = 0;
  base = -1;
}
void BlockTensor::add(const Key& k, int r, int c) {
  keys.push_back(k);
  rows.push_back(r);
  cols.push_back(c);
}
void BlockTensor::finalize() {
  off.resize(keys.size());
  ld = cols;
  col0.assign(keys.size(), 0);
  index.clear();
  index.reserve(keys.size() * 2);
  int64_t n = 0;
  for (size_t i = 0; i < keys.size(); ++i) {
    off[i] = n;
    n += (int64_t)rows[i] * cols[i];
    index[keys[i]] = (int)i;
  }
  nelem = n;
}
void BlockTensor::finalize_panels(const std::vector<int>& panel, const std::vector<int>& order) {
  const size_t n = keys.size();
  off.assign(n, 0);
  ld.assign(n, 0);
  col0.assign(n, 0);
  int np = 0;
  for (int p : panel) np = std::max(np, p + 1);
  std::vector<std::vector<int>> mem(np);
  for (size_t i = 0; i < n; ++i) mem[panel[i]].push_back((int)i);
  int64_t base_ = 0;
  for (int p = 0; p < np; ++p) {
    std::vector<int>& m = mem[p];
    if (m.empty()) continue;
    std::sort(m.begin(), m.end(), [&](int a, int b) { return order[a] != order[b] ? order[a] < order[b] : a < b; });
    int w = 0;
    for (int i : m) {
      if (rows[i] != rows[m[0]]) throw std::runtime_error("fused layout: blocks of a panel differ in row count");
      col0[i] = w;
      w += cols[i];
    }
    for (int i : m) {
      ld[i] = w;
      off[i] = base_ + col0[i];
    }
    base_ += (int64_t)rows[m[0]] * w;
  }
  nelem = base_;
  index.clear();
  index.reserve(n * 2);
  for (size_t i = 0; i < n; ++i) index[keys[i]] = (int)i;
}
int BlockTensor::find(const Key& k) const {
  auto it = index.find(k);
  return it == index.end() ? -1 : it->second;
}

static inline Sector key_sector(const Key& k, int pos) { return Sector{k[pos], k[pos + 1]}; }

// labels c with a (x) s -> c
static inline int fuse(Sector a, int s, Sector out[2]) {
  int n = 0;
  const int ts = SITE_TJ[s];
  for (int tc = std::abs(a.tj - ts); tc <= a.tj + ts; tc += 2) out[n++] = Sector{a.q + SITE_Q[s], tc};
  return n;
}

// column rank of the (s2, b) group inside a fused row panel: s2 in the order 0, 2, 1, then b by (q, tj)
static inline int theta_col_rank(int s2, int bq, int btj) {
  static const int perm[4] = {0, 2, 1, 3};  // SU2: s2 = 0, 2, 1; U1U1: plain order apart from that swap
  return (perm[s2] << 24) + ((bq + 4096) << 11) + btj;
}

void layout_site(const Bond& bl, const Bond& br, BlockTensor& out) {
  out.clear();
  out.nlab = 5;
  std::vector<std::pair<Key, std::pair<int, int>>> v;
  for (size_t ia = 0; ia < bl.sec.size(); ++ia)
    for (int s = 0; s < sym().ns; ++s) {
      Sector cs[2];
      int n = fuse(bl.sec[ia], s, cs);
      for (int j = 0; j < n; ++j) {
        int ic = br.find(cs[j]);
        if (ic >= 0) v.push_back({key_site(bl.sec[ia], s, cs[j]), {bl.d[ia], br.d[ic]}});
      }
    }
  std::sort(v.begin(), v.end(), [](const auto& x, const auto& y) { return x.first < y.first; });
  for (auto& e : v) out.add(e.first, e.second.first, e.second.second);
  out.finalize();
}

void layout_theta(const Bond& bl, const Bond& br, BlockTensor& out) {
  out.clear();
  out.nlab = 8;
  std::vector<std::pair<Key, std::pair<int, int>>> v;
  for (size_t ia = 0; ia < bl.sec.size(); ++ia)
    for (int s1 = 0; s1 < sym().ns; ++s1) {
      Sector cs[2];
      int nc = fuse(bl.sec[ia], s1, cs);
      for (int j = 0; j < nc; ++j)
        for (int s2 = 0; s2 < sym().ns; ++s2) {
          Sector bs[2];
          int nb = fuse(cs[j], s2, bs);
          for (int l = 0; l < nb; ++l) {
            int ib = br.find(bs[l]);
            if (ib >= 0) v.push_back({key_theta(bl.sec[ia], s1, cs[j], s2, bs[l]), {bl.d[ia], br.d[ib]}});
          }
        }
    }
  std::sort(v.begin(), v.end(), [](const auto& x, const auto& y) { return x.first < y.first; });
  for (auto& e : v) out.add(e.first, e.second.first, e.second.second);
  // Fused layout: for every middle label c the blocks form ONE row-major matrix
  // theta_c[(a,s1,alpha), (s2,b,beta)] -- the matrix M_c of the SVD split (H8) -- with row groups in (a,s1)
  // order; column groups ordered s2 = 0, 2, 1 (then b), so that the columns the stage-1 intermediates of
  // w_m = P (s2 in {0,2}) and w_m = M (s2 in {2,1}) need are contiguous.  A row group is a "panel".
  const size_t n = out.keys.size();
  std::vector<std::array<int, 5>> pk(n);  // (c.q, c.tj, a.q, a.tj, s1)
  for (size_t i = 0; i < n; ++i) {
    const Key& k = out.keys[i];
    pk[i] = {k[3], k[4], k[0], k[1], k[2]};
  }
  std::vector<std::array<int, 5>> uniq(pk);
  std::sort(uniq.begin(), uniq.end());
  uniq.erase(std::unique(uniq.begin(), uniq.end()), uniq.end());
  std::vector<int> panel(n), order(n);
  for (size_t i = 0; i < n; ++i) {
    const Key& k = out.keys[i];
    panel[i] = (int)(std::lower_bound(uniq.begin(), uniq.end(), pk[i]) - uniq.begin());
    order[i] = theta_col_rank(k[5], k[6], k[7]);
  }
  out.finalize_panels(panel, order);
}

// ----------------------------------------------------------------------------- reduced MPO (F-2, F-3)
void mpo_site_table(int site, double t_h, double U, MpoSite& W) {
  for (int a = 0; a < MAX_NW; ++a)
    for (int b = 0; b < MAX_NW; ++b) {
      W.rank2[a][b] = -1;
      for (int i = 0; i < MAX_NS; ++i)
        for (int j = 0; j < MAX_NS; ++j) W.val[a][b][i][j] = 0.0;
    }
  if (sym().id == 1) {
    // U(1) x U(1): Eq. (1) PAPER.md:26-30 literally.  Local states 0 |0>, 1 |up>, 2 |dn>, 3 |updn> = c+_up c+_dn |0>;
    // Jordan-Wigner in mode order 1up, 1dn, 2up, ...:  c+_{i s} c_{i+1 s} = (c+_s P)_i (c_s)_{i+1},
    // c+_{i+1 s} c_{i s} = -(c_s P)_i (c+_s)_{i+1} with P = (-1)^n, so that
    //   row 0 (start): I, c+_up P, c+_dn P, c_up P, c_dn P, U n_up n_dn;  column 5 (close): -t c_up, -t c_dn, +t c+_up, +t c+_dn;  I.
    // Non-zero elements <s'|op|s>: c+_up: (1,0) = 1, (3,2) = 1;  c+_dn: (2,0) = 1, (3,1) = -1;  c = transposes.
    const double P[4] = {1.0, -1.0, -1.0, 1.0};
    double cu[4][4] = {}, cd[4][4] = {};  // creation operators [s'][s]
    cu[1][0] = 1.0;
    cu[3][2] = 1.0;
    cd[2][0] = 1.0;
    cd[3][1] = -1.0;
    for (int w = 0; w < 6; ++w) W.rank2[0][w] = 0;
    for (int w = 1; w < 6; ++w) W.rank2[w][5] = 0;
    for (int sp = 0; sp < 4; ++sp)
      for (int s = 0; s < 4; ++s) {
        W.val[0][0][sp][s] = W.val[5][5][sp][s] = sp == s ? 1.0 : 0.0;
        W.val[0][1][sp][s] = cu[sp][s] * P[s];      // c+_up P
        W.val[0][2][sp][s] = cd[sp][s] * P[s];      // c+_dn P
        W.val[0][3][sp][s] = cu[s][sp] * P[s];      // c_up P
        W.val[0][4][sp][s] = cd[s][sp] * P[s];      // c_dn P
        W.val[1][5][sp][s] = -t_h * cu[s][sp];      // -t c_up
        W.val[2][5][sp][s] = -t_h * cd[s][sp];      // -t c_dn
        W.val[3][5][sp][s] = +t_h * cu[sp][s];      // +t c+_up
        W.val[4][5][sp][s] = +t_h * cd[sp][s];      // +t c+_dn
      }
    W.val[0][5][3][3] = U;  // U n_up n_dn
    return;
  }
  const double eps = (site % 2 == 0) ? 1.0 : -1.0;  // eps_i = (-1)^i, 0-based (reading A-3)
  const double eps_prev = -eps;
  const double r2 = std::sqrt(2.0);
  // identity and (U/2) P_D, rank 0
  W.rank2[0][0] = 0;
  W.rank2[3][3] = 0;
  W.rank2[0][3] = 0;
  for (int s = 0; s < 3; ++s) W.val[0][0][s][s] = W.val[3][3][s][s] = 1.0;
  W.val[0][3][2][2] = 0.5 * U;
  // opening operators Psi^+ P (S->P) and Psi^- P (S->M), rank 1/2
  W.rank2[0][1] = 1;
  W.val[0][1][0][2] = -r2;
  W.val[0][1][2][1] = -eps;
  W.rank2[0][2] = 1;
  W.val[0][2][1][2] = -r2;
  W.val[0][2][2][0] = +eps;
  // closing operators: P->F carries -t eps_{i-1} sqrt2 Psi^-, M->F carries +t eps_{i-1} sqrt2 Psi^+
  W.rank2[1][3] = 1;
  W.val[1][3][1][2] = -t_h * eps_prev * r2 * (-r2);
  W.val[1][3][2][0] = -t_h * eps_prev * r2 * (-eps);
  W.rank2[2][3] = 1;
  W.val[2][3][0][2] = +t_h * eps_prev * r2 * (-r2);
  W.val[2][3][2][1] = +t_h * eps_prev * r2 * (+eps);
}

// ----------------------------------------------------------------------------- stage assembly
// Unit decomposition: every output block is cut into warp units of
// (8 mt) x (8 nt) elements, mt * nt <= GEMM_MAX_SUBTILES, chosen per block so that (i) only the
// last row / column of 8x8 sub-tiles is padded, (ii) one unit issues at most ~GEMM_UNIT_DMMA_CAP
// DMMAs (long-K blocks get smaller units so that there are enough of them to fill 148 SMs), and
// (iii) the number of operand fragments loaded per DMMA is minimal under (i) and (ii).
static const int GEMM_MAX_SUBTILES = 16;
static const int GEMM_MAX_DIM = 8;
static const int GEMM_UNIT_DMMA_CAP = 3072;

static void emit_units(Stage& st) {
  struct UW {
    GemmUnit u;
    int64_t work;
  };
  std::vector<UW> v;
  v.reserve(st.mouts.size() * 2);
  st.dmma_padded = 0;
  // The per-unit cap only exists to create enough units for 148 SMs x 8 resident warps; when the
  // stage is large (chi >~ 8000) full 16-sub-tile units are plentiful and the cap is lifted
  // (measured at chi = 16384: 31.0 TFLOP/s uncapped vs 20.9 with the cap of 3072).
  int64_t total16 = 0;
  for (const GemmOut& o : st.mouts) total16 += (int64_t)4 * ((o.M + 7) / 8) * ((o.N + 7) / 8) * o.steps;
  // Small stages (one-site and zero-site applies, environment updates at chi = 4096: well under a million DMMAs)
  // want smaller units still: a unit should not be longer than the fair share of one of the 1184 warp slots,
  // else the stage lasts as long as its few heaviest units (one-site apply at chi = 4096: 82 -> 71 us with the
  // cap lowered from 3072 to 1024, the chi = 1024 apply 61 -> 32 us with 256, while the two-site apply at chi = 4096,
  // 4.1e6 DMMAs per stage, is fastest at 3072).
  const int64_t cap_floor = 256;
  const int64_t fair = 2 * (total16 / (148 * 8));  // twice the even share: measured best at chi = 1024, 4096 (one- and two-site)
  const int64_t base_cap = std::min<int64_t>(GEMM_UNIT_DMMA_CAP, std::max<int64_t>(cap_floor, fair));
  const int64_t cap = std::max<int64_t>(base_cap, total16 / (148 * 8 * 6));
  for (size_t oi = 0; oi < st.mouts.size(); ++oi) {
    const GemmOut& o = st.mouts[oi];
    if (o.M <= 0 || o.N <= 0) continue;
    const int M8 = (o.M + 7) / 8, N8 = (o.N + 7) / 8;
    const int s_t = (int)std::min<int64_t>(GEMM_MAX_SUBTILES, std::max<int64_t>(2, cap / std::max(1, 4 * o.steps)));
    int best_h = 1, best_w = 1;
    long best_cost = -1, best_units = 0;
    for (int h = 1; h <= std::min(GEMM_MAX_DIM, M8); ++h) {
      const int g = (M8 + h - 1) / h, hm = (M8 + g - 1) / g;
      const int wmax = std::min(GEMM_MAX_DIM, s_t / hm);
      if (wmax < 1) continue;
      const int nu = (N8 + wmax - 1) / wmax;
      const long cost = (long)nu * M8 + (long)g * N8, nun = (long)nu * g;  // fragments loaded per k-step
      if (best_cost < 0 || cost < best_cost || (cost == best_cost && nun < best_units)) {
        best_cost = cost;
        best_units = nun;
        best_h = hm;
        best_w = wmax;
      }
    }
    const int g = (M8 + best_h - 1) / best_h, nu = (N8 + best_w - 1) / best_w;
    int m8 = 0;
    for (int i = 0; i < g; ++i) {
      const int h = M8 / g + (i < M8 % g ? 1 : 0);
      int n8 = 0;
      for (int j = 0; j < nu; ++j) {
        const int w = N8 / nu + (j < N8 % nu ? 1 : 0);
        UW x;
        x.u = GemmUnit{o.c_off, o.ldc, o.M, o.N, o.seg_begin, o.seg_end, o.steps, m8 * 8, n8 * 8, h * 16 + w, (int)oi,
                         o.seg_end > o.seg_begin ? st.segs[o.seg_begin] : GemmSeg{0, 0, 0, 0, 0, 0, 0, 0, 0.0}};
        x.work = (int64_t)h * w * std::max(1, o.steps);
        st.dmma_padded += 4 * (int64_t)h * w * o.steps;
        v.push_back(x);
        n8 += w;
      }
      m8 += h;
    }
  }
  // heaviest first: the hardware CTA scheduler (one unit per one-warp CTA) then balances greedily.
  // (work, emission index) pairs are sorted, not the 96-byte descriptors; equal work keeps emission order.
  std::vector<std::pair<int64_t, int>> ord(v.size());
  for (size_t i = 0; i < v.size(); ++i) ord[i] = {-v[i].work, (int)i};
  std::sort(ord.begin(), ord.end());
  st.units.clear();
  st.units.reserve(v.size());
  for (auto& o : ord) st.units.push_back(v[o.second].u);
}

// Tile decomposition for the warp-specialised kernel (zgemm_ws.cu).  Every (merged) output is cut into a grid
// of tiles of h x w sub-tiles of 8 x 8 (h, w <= 8; a group of 2 x 2 warps takes one tile, every warp at most
// 4 x 4 sub-tiles), as evenly as the sub-tile counts allow -- tile SHAPES stay as large as the block allows,
// because a warp's efficiency rests on its register tile.  Balance comes from splitting along k instead: a
// tile heavier than the cap (a fraction of the even share of one of the 2 x 148 groups) is cut into parts at
// chunk boundaries (16 k); all parts but the one that starts at k = 0 leave their accumulators in a scratch
// slot, and that one adds them in slot order and stores the block (fixed order: deterministic).  In the queue
// the parts of a tile come before its finishing part, so a finisher never waits for work not yet handed out.
void emit_ws_tiles(Stage& st) {
  st.tiles.clear();
  st.n_slots = 0;
  st.mout_tiles.assign(st.mouts.size(), 0);
  int64_t total = 0;
  for (const GemmOut& o : st.mouts) total += (int64_t)4 * ((o.M + 7) / 8) * ((o.N + 7) / 8) * std::max(1, o.steps);
  // cap = the even share of one group: measured at chi = 4096 / 8192, smaller caps (more, k-split tiles) cost
  // more in partial-sum traffic and tile switches than they gain in balance
  const int64_t cap = std::max<int64_t>(2048, total / 296);
  struct TW {
    WsTile t;
    int64_t key;  // sort key: work of the heaviest part of the (split) tile
    int uid, rank;
  };
  std::vector<TW> v;
  int uid = 0;
  std::vector<int> cseg, ck;  // chunk -> (segment, k offset)
  for (const GemmOut& o : st.mouts) {
    if (o.M <= 0 || o.N <= 0) continue;
    const int M8 = (o.M + 7) / 8, N8 = (o.N + 7) / 8;
    const int gh = (M8 + 7) / 8, gw = (N8 + 7) / 8;
    cseg.clear();
    ck.clear();
    for (int sgi = o.seg_begin; sgi < o.seg_end; ++sgi)
      for (int k = 0; k < st.segs[sgi].K; k += 16) {
        cseg.push_back(sgi);
        ck.push_back(k);
      }
    const int nch = (int)cseg.size();
    int m8 = 0;
    for (int i = 0; i < gh; ++i) {
      const int h = M8 / gh + (i < M8 % gh ? 1 : 0);
      int n8 = 0;
      for (int j = 0; j < gw; ++j) {
        const int w = N8 / gw + (j < N8 % gw ? 1 : 0);
        if (h > 0 && w > 0) {
          const int64_t work = (int64_t)4 * h * w * std::max(1, o.steps);
          int P = (int)std::min<int64_t>(8, (work + cap - 1) / cap);
          P = std::max(1, std::min(P, nch / 2));  // at least two chunks per part
          WsTile base = WsTile{o.c_off, o.ldc, o.M, o.N, m8 * 8, n8 * 8, h, w, o.seg_begin, o.seg_end, o.steps,
                               o.seg_end > o.seg_begin ? st.segs[o.seg_begin] : GemmSeg{0, 0, 0, 0, 0, 0, 0, 0, 0.0},
                               0, 1 << 30, 0, 0, 0, 0, 0, 0};
          base.stage_sig = ((int)(&o - &st.mouts[0]) + 1) << 1;  // stage bit set by link_stages
          const int slot0 = st.n_slots;
          int64_t key = 0;
          std::vector<TW> parts;
          for (int p = 0; p < P; ++p) {
            const int cb = (int)((int64_t)nch * p / P), ce = (int)((int64_t)nch * (p + 1) / P);
            TW x;
            x.t = base;
            int steps = o.steps;
            if (P > 1) {
              x.t.seg_begin = cseg[cb];
              x.t.k_begin = ck[cb];
              x.t.seg_end = cseg[ce - 1] + 1;
              x.t.k_end = ck[ce - 1] + 16;  // clipped to the segment's K by the producer
              x.t.first = st.segs[x.t.seg_begin];
              steps = 0;
              for (int c = cb; c < ce; ++c) steps += (std::min(16, st.segs[cseg[c]].K - ck[c]) + 3) / 4;
              x.t.steps = steps;
              if (p == 0) {
                x.t.kind = 0;
                x.t.slot = slot0;
                x.t.nparts = P - 1;
              } else {
                x.t.kind = 1;
                x.t.slot = slot0 + p - 1;
                x.t.nparts = 0;
              }
            }
            x.t.nparts |= std::max(1, ce - cb) << 8;  // chunks of this part (a block without segments has one)
            // arrangement of the group's four warps on the tile: the one whose largest part is smallest
            // (0: 2 x 2 quadrants, 1: four column strips, 2: four row strips; a part is at most 16 sub-tiles)
            const int part22 = ((h + 1) / 2) * ((w + 1) / 2);
            const int partc = h * ((w + 3) / 4), partr = ((h + 3) / 4) * w;
            int arr = 0, part = part22;
            if ((w + 3) / 4 <= 2 && partc < part) {
              arr = 1;
              part = partc;
            }
            if ((h + 3) / 4 <= 2 && partr < part) {
              arr = 2;
              part = partr;
            }
            x.t.kind |= arr << 2;
            // a tile lasts as long as its largest part
            key = std::max<int64_t>(key, (int64_t)part * std::max(1, steps));
            x.uid = uid;
            x.rank = p == 0 ? P : p;  // the finishing part (p = 0) goes last
            parts.push_back(x);
          }
          if (P > 1) st.n_slots += P - 1;
          ++st.mout_tiles[&o - &st.mouts[0]];  // one storing tile (the finishing part of a split one)
          for (TW& x : parts) {
            x.key = key;
            v.push_back(x);
          }
          ++uid;
        }
        n8 += w;
      }
      m8 += h;
    }
  }
  std::vector<int> ord(v.size());
  for (size_t i = 0; i < v.size(); ++i) ord[i] = (int)i;
  std::sort(ord.begin(), ord.end(), [&](int a, int b) {
    if (v[a].key != v[b].key) return v[a].key > v[b].key;
    if (v[a].uid != v[b].uid) return v[a].uid < v[b].uid;
    return v[a].rank < v[b].rank;
  });
  st.tiles.reserve(v.size());
  for (int i : ord) st.tiles.push_back(v[i].t);
}

// Outputs that lie side by side in one row panel (N direction) or one below the other (M direction) and
// whose segment lists describe the same GEMM on adjacent operand columns / rows are ONE wider / taller GEMM:
// the merged output keeps the segment list of its first member (the kernel addresses operands by offset and
// stride only, so columns n >= N_first simply run on into the neighbour block).  The canonical per-block
// lists (outs, segs, t_*) are untouched; only the unit decomposition uses mouts.
static void merge_outs(Stage& st, int64_t lhs_nelem, int64_t rhs_nelem) {
  st.mouts.clear();
  st.mouts.reserve(st.outs.size());
  std::vector<std::vector<int>> members;  // original output blocks of every entry of mouts
  for (size_t oi = 0; oi < st.outs.size(); ++oi) {
    const GemmOut& o = st.outs[oi];
    if (o.M > 0 && o.N > 0) {
      st.mouts.push_back(o);
      members.push_back(std::vector<int>(1, (int)oi));
    }
  }
  for (int dir = 0; dir < 2; ++dir) {  // 0: N direction, 1: M direction
    std::vector<GemmOut>& v = st.mouts;
    std::unordered_map<int64_t, int> by_off;
    by_off.reserve(v.size() * 2);
    for (size_t i = 0; i < v.size(); ++i) by_off[v[i].c_off] = (int)i;
    std::vector<int> ord(v.size());
    for (size_t i = 0; i < v.size(); ++i) ord[i] = (int)i;
    std::sort(ord.begin(), ord.end(), [&](int a, int b) { return v[a].c_off < v[b].c_off; });
    std::vector<char> dead(v.size(), 0);
    for (int i : ord) {
      if (dead[i]) continue;
      GemmOut& o = v[i];
      for (;;) {
        const int64_t next = dir == 0 ? o.c_off + o.N : o.c_off + (int64_t)o.M * o.ldc;
        auto it = by_off.find(next);
        if (it == by_off.end()) break;
        const int j = it->second;
        if (j == i || dead[j]) break;
        const GemmOut& p = v[j];
        const int ns = o.seg_end - o.seg_begin;
        if (p.ldc != o.ldc || p.seg_end - p.seg_begin != ns || ns == 0) break;
        if (dir == 0 ? (p.M != o.M || p.col0 != o.col0 + o.N) : (p.N != o.N || p.col0 != o.col0)) break;
        bool ok = true;
        for (int t = 0; t < ns && ok; ++t) {
          const GemmSeg& a = st.segs[o.seg_begin + t];
          const GemmSeg& b = st.segs[p.seg_begin + t];
          ok = a.K == b.K && a.alpha == b.alpha && a.a_sm == b.a_sm && a.a_sk == b.a_sk && a.b_sk == b.b_sk &&
               a.b_sn == b.b_sn;
          if (dir == 0) ok = ok && a.a_off == b.a_off && b.b_off == a.b_off + (int64_t)o.N * a.b_sn;
          else ok = ok && b.b_off == a.b_off && b.a_off == a.a_off + (int64_t)o.M * a.a_sm;
        }
        if (!ok) break;
        if (dir == 0) o.N += p.N;
        else o.M += p.M;
        members[i].insert(members[i].end(), members[j].begin(), members[j].end());
        dead[j] = 1;
      }
    }
    std::vector<GemmOut> kept;
    std::vector<std::vector<int>> keptm;
    kept.reserve(v.size());
    for (size_t i = 0; i < v.size(); ++i)
      if (!dead[i]) {
        kept.push_back(v[i]);
        keptm.push_back(std::move(members[i]));
      }
    v.swap(kept);
    members.swap(keptm);
  }
  st.out_mout.assign(st.outs.size(), -1);
  for (size_t m = 0; m < members.size(); ++m)
    for (int oi : members[m]) st.out_mout[oi] = (int)m;
  // every merged GEMM stays inside its operand tensors (same proof as for the single blocks)
  for (const GemmOut& o : st.mouts)
    for (int t = o.seg_begin; t < o.seg_end; ++t) {
      const GemmSeg& sg = st.segs[t];
      if (sg.K <= 0) continue;
      const int64_t a_last = sg.a_off + (int64_t)(o.M - 1) * sg.a_sm + (int64_t)(sg.K - 1) * sg.a_sk;
      const int64_t b_last = sg.b_off + (int64_t)(sg.K - 1) * sg.b_sk + (int64_t)(o.N - 1) * sg.b_sn;
      if (a_last >= lhs_nelem || b_last >= rhs_nelem) throw std::runtime_error("task list: merged operand exceeds its tensor");
    }
}

// Joint tile queue of two dependent stages for ONE launch of the warp-specialised kernel (WsPair): stage-1 tiles
// (heaviest first), then stage-2 tiles (heaviest first).  A stage-2 tile lists the stage-1 merged outputs that
// hold the blocks its segments read (as lhs, or as rhs when mid_is_rhs2); it may start once each of them has
// collected 4 arrivals (the four warps of a group) per storing tile.
void link_stages(const Stage& st1, const Stage& st2, int mid_is_rhs2, WsPair& pr) {
  pr.tiles.clear();
  pr.segs = st1.segs;
  pr.segs.insert(pr.segs.end(), st2.segs.begin(), st2.segs.end());
  pr.dep_id.clear();
  pr.dep_target.clear();
  pr.n_dep_counters = (int)st1.mouts.size();
  pr.n_slots = st1.n_slots + st2.n_slots;
  pr.conj1 = st1.opA != OPA_N;
  pr.conj2 = st2.opA != OPA_N;
  pr.tiles.reserve(st1.tiles.size() + st2.tiles.size());
  for (const WsTile& t : st1.tiles) pr.tiles.push_back(t);  // stage bit 0, sig as emitted
  // dependency list of every stage-2 merged output
  const int nseg1 = (int)st1.segs.size();
  std::vector<int> dbeg(st2.mouts.size(), 0), dcnt(st2.mouts.size(), 0);
  std::vector<std::vector<int>> deps(st2.mouts.size());
  for (size_t o = 0; o < st2.outs.size(); ++o) {
    const int m = st2.out_mout[o];
    if (m < 0) continue;
    for (int t = st2.outs[o].seg_begin; t < st2.outs[o].seg_end; ++t) {
      const int z = mid_is_rhs2 ? st2.t_rhs[t] : st2.t_lhs[t];
      const int zm = st1.out_mout[z];
      if (zm >= 0) deps[m].push_back(zm);
    }
  }
  for (size_t m = 0; m < deps.size(); ++m) {
    std::sort(deps[m].begin(), deps[m].end());
    deps[m].erase(std::unique(deps[m].begin(), deps[m].end()), deps[m].end());
    dbeg[m] = (int)pr.dep_id.size();
    dcnt[m] = (int)deps[m].size();
    for (int zm : deps[m]) {
      pr.dep_id.push_back(zm);
      pr.dep_target.push_back(4u * (unsigned)st1.mout_tiles[zm]);
    }
  }
  for (const WsTile& t0 : st2.tiles) {
    WsTile t = t0;
    const int m = (t.stage_sig >> 1) - 1;
    t.stage_sig = 1;  // stage 2, nothing to signal
    t.seg_begin += nseg1;
    t.seg_end += nseg1;
    t.slot += st1.n_slots;
    t.dep_begin = dbeg[m];
    t.dep_count = dcnt[m];
    pr.tiles.push_back(t);
  }
}

// The same for the warp-unit form: ONE launch whose grid is the stage-1 units followed by the stage-2 units (each
// list heaviest first).  A stage-1 unit raises the counter of the merged output it tiles when its stores are
// done; a stage-2 unit waits until every stage-1 output its segments read has collected one arrival per unit
// that tiles it.  One-warp CTAs are dispatched in index order, so every stage-1 unit has started before a
// stage-2 unit can occupy a warp slot: waiting cannot deadlock.
void link_units(const Stage& st1, const Stage& st2, int mid_is_rhs2, UnitPair& pr) {
  const int nseg1 = (int)st1.segs.size();
  pr.segs = st1.segs;
  pr.segs.insert(pr.segs.end(), st2.segs.begin(), st2.segs.end());
  pr.n1 = (int)st1.units.size();
  pr.n_dep_counters = (int)st1.mouts.size();
  pr.conj1 = st1.opA != OPA_N;
  pr.conj2 = st2.opA != OPA_N;
  pr.units.clear();
  pr.link.clear();
  pr.dep_id.clear();
  pr.dep_target.clear();
  pr.units.reserve(st1.units.size() + st2.units.size());
  std::vector<unsigned> tiled(st1.mouts.size(), 0);  // units per stage-1 merged output (GemmUnit::pad = its index)
  for (const GemmUnit& u : st1.units) ++tiled[u.pad];
  for (const GemmUnit& u : st1.units) {
    pr.units.push_back(u);
    pr.link.push_back(UnitLink{0, u.pad, 0, 0});
  }
  std::vector<std::vector<int>> deps(st2.mouts.size());
  for (size_t o = 0; o < st2.outs.size(); ++o) {
    const int m = st2.out_mout[o];
    if (m < 0) continue;
    for (int t = st2.outs[o].seg_begin; t < st2.outs[o].seg_end; ++t) {
      const int z = mid_is_rhs2 ? st2.t_rhs[t] : st2.t_lhs[t];
      const int zm = st1.out_mout[z];
      if (zm >= 0) deps[m].push_back(zm);
    }
  }
  std::vector<int> dbeg(deps.size(), 0), dcnt(deps.size(), 0);
  for (size_t m = 0; m < deps.size(); ++m) {
    std::sort(deps[m].begin(), deps[m].end());
    deps[m].erase(std::unique(deps[m].begin(), deps[m].end()), deps[m].end());
    dbeg[m] = (int)pr.dep_id.size();
    dcnt[m] = (int)deps[m].size();
    for (int zm : deps[m]) {
      pr.dep_id.push_back(zm);
      pr.dep_target.push_back(tiled[zm]);
    }
  }
  for (const GemmUnit& u0 : st2.units) {
    GemmUnit u = u0;
    u.seg_begin += nseg1;
    u.seg_end += nseg1;
    pr.units.push_back(u);
    pr.link.push_back(UnitLink{1, -1, dbeg[u0.pad], dcnt[u0.pad]});
  }
}

void finalize_stage(Stage& st, const BlockTensor& out, const BlockTensor& lhs, const BlockTensor& rhs) {
  const size_t nt = st.t_out.size();
  st.outs.resize(out.keys.size());
  st.segs.resize(nt);
  st.flops = 0;
  const bool scaled = st.t_scale.size() == nt && nt > 0;
  size_t t = 0;
  for (size_t o = 0; o < out.keys.size(); ++o) {
    GemmOut& go = st.outs[o];
    go.c_off = out.off[o];
    go.M = out.rows[o];
    go.N = out.cols[o];
    go.ldc = out.ld[o];
    go.col0 = out.col0[o];
    go.steps = 0;
    go.seg_begin = (int)t;
    while (t < nt && st.t_out[t] == (int)o) {
      const int l = st.t_lhs[t], r = st.t_rhs[t];
      GemmSeg& sg = st.segs[t];
      sg.a_off = lhs.off[l];
      sg.b_off = rhs.off[r];
      sg.pad = 0;
      sg.alpha = scaled ? st.t_alpha[t] * st.t_scale[t] : st.t_alpha[t];
      int M, K, K2, N;
      if (st.opA == OPA_H) {  // stored K x M
        M = lhs.cols[l];
        K = lhs.rows[l];
        sg.a_sm = 1;
        sg.a_sk = lhs.ld[l];
      } else {  // stored M x K
        M = lhs.rows[l];
        K = lhs.cols[l];
        sg.a_sm = lhs.ld[l];
        sg.a_sk = 1;
      }
      if (st.opB == OPB_T) {  // stored N x K
        N = rhs.rows[r];
        K2 = rhs.cols[r];
        sg.b_sk = 1;
        sg.b_sn = rhs.ld[r];
      } else {  // stored K x N
        N = rhs.cols[r];
        K2 = rhs.rows[r];
        sg.b_sk = rhs.ld[r];
        sg.b_sn = 1;
      }
      if (M != go.M || N != go.N || K != K2) throw std::runtime_error("task list: block shapes do not match");
      sg.K = K;
      // The kernel reads op(A)(m, k) and op(B)(k, n) only for m < M, n < N, k < K (rows, columns and
      // k positions beyond are clamped to the last valid one), so proving the extreme element of each
      // operand inside its tensor proves every copy of the kernel in bounds.
      if (K > 0) {
        const int64_t a_last = sg.a_off + (int64_t)(M - 1) * sg.a_sm + (int64_t)(K - 1) * sg.a_sk;
        const int64_t b_last = sg.b_off + (int64_t)(K - 1) * sg.b_sk + (int64_t)(N - 1) * sg.b_sn;
        if (sg.a_off < 0 || sg.b_off < 0 || a_last >= lhs.nelem || b_last >= rhs.nelem)
          throw std::runtime_error("task list: operand block exceeds its tensor");
      }
      go.steps += (K + 3) / 4;
      st.flops += (int64_t)8 * M * N * K;
      ++t;
    }
    go.seg_end = (int)t;
    if (go.c_off < 0 || go.c_off + (int64_t)(go.M - 1) * go.ldc + go.N > out.nelem)
      throw std::runtime_error("task list: output block exceeds its tensor");
  }
  if (t != nt) throw std::runtime_error("task list: tasks not sorted by output id");
  merge_outs(st, lhs.nelem, rhs.nelem);
  emit_units(st);
  // the tile list of the warp-specialised form is emitted on demand (emit_ws_tiles): only two-site plans in its size
  // window use it, and every stage of a sweep passes through here
  st.tiles.clear();
  st.n_slots = 0;
}

namespace {
struct RawTask {
  Key out;      // output block key
  Key order;    // segment sort key
  int lhs, rhs;
  double alpha;
  double scale = 1.0;  // factor on alpha outside the canonical list (weights of the vector gauge)
};

// the first seven ints of an `order` key packed so that integer order == lexicographic order
// (each field offset by 64 into 8 bits); false if a field does not fit
static bool pack_order(const Key& k, uint64_t& packed) {
  packed = 0;
  for (int i = 0; i < 7; ++i) {
    const int v = k[i] + 64;
    if (v < 0 || v > 255) return false;
    packed = (packed << 8) | (uint64_t)v;
  }
  for (int i = 7; i < 12; ++i)
    if (k[i] != 0) return false;
  return true;
}

// fill st.t_* from raw tasks in canonical order (output block, then `order`); `out` must already contain
// every key that occurs.  The output index of `out` is ascending in the key, so sorting (index, packed
// order) pairs gives the same sequence as sorting the 96-byte keys themselves.
void tasks_to_stage(std::vector<RawTask>& raw, const BlockTensor& out, Stage& st) {
  struct Ref {
    int o;
    uint64_t ord;
    int idx;
  };
  std::vector<Ref> refs(raw.size());
  bool packed_ok = true;
  for (size_t i = 0; i < raw.size(); ++i) {
    refs[i].o = out.find(raw[i].out);
    if (refs[i].o < 0) throw std::runtime_error("task list: output key missing from layout");
    refs[i].idx = (int)i;
    packed_ok = packed_ok && pack_order(raw[i].order, refs[i].ord);
  }
  if (packed_ok) {
    std::sort(refs.begin(), refs.end(), [](const Ref& a, const Ref& b) {
      return a.o != b.o ? a.o < b.o : (a.ord != b.ord ? a.ord < b.ord : a.idx < b.idx);
    });
  } else {
    std::sort(refs.begin(), refs.end(), [&](const Ref& a, const Ref& b) {
      if (a.o != b.o) return a.o < b.o;
      if (raw[a.idx].order != raw[b.idx].order) return raw[a.idx].order < raw[b.idx].order;
      return a.idx < b.idx;
    });
  }
  st.t_out.clear();
  st.t_lhs.clear();
  st.t_rhs.clear();
  st.t_alpha.clear();
  st.t_out.reserve(raw.size());
  st.t_lhs.reserve(raw.size());
  st.t_rhs.reserve(raw.size());
  st.t_alpha.reserve(raw.size());
  st.t_scale.clear();
  bool any_scale = false;
  for (const RawTask& r : raw) any_scale = any_scale || r.scale != 1.0;
  if (any_scale) st.t_scale.reserve(raw.size());
  for (const Ref& f : refs) {
    const RawTask& r = raw[f.idx];
    st.t_out.push_back(f.o);
    st.t_lhs.push_back(r.lhs);
    st.t_rhs.push_back(r.rhs);
    st.t_alpha.push_back(r.alpha);
    if (any_scale) st.t_scale.push_back(r.scale);
  }
}

// layout from the distinct output keys of raw tasks: rows/cols supplied per task
struct Shape {
  int r, c;
};
void layout_from_tasks(const std::vector<RawTask>& raw, const std::vector<Shape>& shapes, int nlab,
                       BlockTensor& out) {
  std::unordered_map<Key, int, KeyHash> seen;
  seen.reserve(raw.size());
  std::vector<std::pair<Key, Shape>> uniq;
  for (size_t i = 0; i < raw.size(); ++i) {
    auto ins = seen.emplace(raw[i].out, (int)uniq.size());
    if (ins.second) uniq.push_back({raw[i].out, shapes[i]});
    else uniq[ins.first->second].second = shapes[i];
  }
  std::sort(uniq.begin(), uniq.end(),
            [](const std::pair<Key, Shape>& a, const std::pair<Key, Shape>& b) { return a.first < b.first; });
  out.clear();
  out.nlab = nlab;
  for (auto& e : uniq) out.add(e.first, e.second.r, e.second.c);
  out.finalize();
}

// Generic "left contraction" (stage 1 of H1, H3, H4):
//   Z[a',s',c',w' ; rest] = sum_{(w,a,s)} alpha * Lenv[a',w,a] * ket[a,s,c; rest]
// ket keys: (a.q,a.tj,s,c.q,c.tj, rest...) with `nrest` extra ints (0 for one-site, 3 for two-site).
void left_contraction_tasks(const BlockTensor& Lenv, const BlockTensor& ket, const MpoSite& W, int nrest,
                            std::vector<RawTask>& raw, std::vector<Shape>& shapes) {
  std::map<Sector, std::vector<int>> by_a;
  for (size_t i = 0; i < ket.keys.size(); ++i) by_a[key_sector(ket.keys[i], 0)].push_back((int)i);
  raw.clear();
  shapes.clear();
  raw.reserve(4 * ket.keys.size());
  shapes.reserve(4 * ket.keys.size());
  for (size_t e = 0; e < Lenv.keys.size(); ++e) {
    const Key& ek = Lenv.keys[e];
    const Sector ap = key_sector(ek, 0), a = key_sector(ek, 3);
    const int w = ek[2];
    auto it = by_a.find(a);
    if (it == by_a.end()) continue;
    for (int ki : it->second) {
      const Key& kk = ket.keys[ki];
      const int s = kk[2];
      const Sector c = key_sector(kk, 3);
      for (int wp = 0; wp < sym().nw; ++wp) {
        const int tr = W.rank2[w][wp];
        if (tr < 0) continue;
        for (int sp = 0; sp < sym().ns; ++sp) {
          const double wv = W.val[w][wp][sp][s];
          if (wv == 0.0) continue;
          Sector cps[2];
          const int ncp = fuse(ap, sp, cps);
          for (int j = 0; j < ncp; ++j) {
            const Sector cp = cps[j];
            if (cp.q != c.q + MPO_Q[wp] || !triangle(c.tj, MPO_TK[wp], cp.tj)) continue;
            const double al = coef_left(a.tj, SITE_TJ[s], c.tj, MPO_TK[w], tr, MPO_TK[wp], ap.tj, SITE_TJ[sp], cp.tj) * wv;
            if (std::fabs(al) < ALPHA_ZERO) continue;
            RawTask t;
            t.out = Key{ap.q, ap.tj, sp, cp.q, cp.tj, wp, c.q, c.tj, 0, 0, 0, 0};
            for (int r = 0; r < nrest; ++r) t.out[8 + r] = kk[5 + r];
            t.order = Key{w, a.q, a.tj, s, 0, 0, 0, 0, 0, 0, 0, 0};
            t.lhs = (int)e;
            t.rhs = ki;
            t.alpha = al;
            raw.push_back(t);
            shapes.push_back(Shape{Lenv.rows[e], ket.cols[ki]});
          }
        }
      }
    }
  }
}
void emit_left_contraction(const BlockTensor& Lenv, const BlockTensor& ket, const MpoSite& W, int nrest,
                           BlockTensor& Z, Stage& st) {
  std::vector<RawTask> raw;
  std::vector<Shape> shapes;
  left_contraction_tasks(Lenv, ket, W, nrest, raw, shapes);
  layout_from_tasks(raw, shapes, 8 + nrest, Z);
  st.opA = OPA_N;
  st.opB = OPB_N;
  tasks_to_stage(raw, Z, st);
  finalize_stage(st, Z, Lenv, ket);
}
}  // namespace

// Two-site apply.  The vector is held in the gauge theta~[..b] = sqrt(2 j_b + 1) theta[..b], in
// which the F-6 inner product is the plain Euclidean one: the stage-2 coefficient of an output block b' fed
// from a column block b carries the extra factor sqrt((2 j_b' + 1) / (2 j_b + 1)) in t_scale, outside the
// canonical alpha the tests compare with the oracle.
void emit_heff2(const BlockTensor& Lenv, const BlockTensor& Renv, const BlockTensor& vec, const MpoSite& W1,
                const MpoSite& W2, BlockTensor& Z, Stage& st1, Stage& st2) {
  std::vector<RawTask> raw1;
  std::vector<Shape> shapes1;
  left_contraction_tasks(Lenv, vec, W1, 3, raw1, shapes1);
  BlockTensor Zall;
  layout_from_tasks(raw1, shapes1, 11, Zall);
  std::map<Sector, std::vector<int>> by_b;
  for (size_t i = 0; i < Renv.keys.size(); ++i) by_b[key_sector(Renv.keys[i], 3)].push_back((int)i);
  std::vector<RawTask> raw;
  std::vector<int> raw_z;  // index into Zall of each stage-2 task's intermediate
  raw.reserve(2 * Zall.keys.size());
  std::vector<char> used(Zall.keys.size(), 0);
  for (size_t z = 0; z < Zall.keys.size(); ++z) {
    const Key& zk = Zall.keys[z];  // a'(0,1) s1'(2) c'(3,4) wm(5) c(6,7) s2(8) b(9,10)
    const Sector ap = key_sector(zk, 0), cp = key_sector(zk, 3), c = key_sector(zk, 6), b = key_sector(zk, 9);
    const int s1p = zk[2], wm = zk[5], s2 = zk[8];
    auto it = by_b.find(b);
    if (it == by_b.end()) continue;
    for (int ri : it->second) {
      const Key& rk = Renv.keys[ri];
      const Sector bp = key_sector(rk, 0);
      const int wr = rk[2];
      const int tr = W2.rank2[wm][wr];
      if (tr < 0) continue;
      for (int s2p = 0; s2p < sym().ns; ++s2p) {
        const double wv = W2.val[wm][wr][s2p][s2];
        if (wv == 0.0) continue;
        const Key ok = key_theta(ap, s1p, cp, s2p, bp);
        if (vec.find(ok) < 0) continue;
        const double al = coef_left(c.tj, SITE_TJ[s2], b.tj, MPO_TK[wm], tr, MPO_TK[wr], cp.tj, SITE_TJ[s2p], bp.tj) * wv;
        if (std::fabs(al) < ALPHA_ZERO) continue;
        RawTask t;
        t.out = ok;
        t.order = Key{c.q, c.tj, s2, b.q, b.tj, wm, wr, 0, 0, 0, 0, 0};
        t.lhs = -1;
        t.rhs = ri;
        t.alpha = al;
        t.scale = std::sqrt((double)(bp.tj + 1) / (double)(b.tj + 1));
        raw.push_back(t);
        raw_z.push_back((int)z);
        used[z] = 1;
      }
    }
  }
  // reading A-17: an intermediate block that no stage-2 task reads is not formed (no task, no storage, no flops)
  {
    std::vector<RawTask> keep1;
    std::vector<Shape> keeps;
    keep1.reserve(raw1.size());
    keeps.reserve(raw1.size());
    for (size_t i = 0; i < raw1.size(); ++i) {
      const int z = Zall.find(raw1[i].out);
      if (z >= 0 && used[z]) {
        keep1.push_back(raw1[i]);
        keeps.push_back(shapes1[i]);
      }
    }
    raw1.swap(keep1);
    shapes1.swap(keeps);
  }
  layout_from_tasks(raw1, shapes1, 11, Z);
  // fused layout of Z: the blocks Z[a',s1',c',w_m; c, (s2,b)] of one (a',s1',c',w_m,c) lie side by side in the
  // column order of the vector, so that stage 1 forms each such row panel with ONE GEMM per segment
  {
    const size_t n = Z.keys.size();
    std::vector<int> panel(n), order(n);
    int np = -1;
    for (size_t i = 0; i < n; ++i) {
      const Key& k = Z.keys[i];
      bool same = i > 0;
      for (int x = 0; same && x < 8; ++x) same = k[x] == Z.keys[i - 1][x];
      if (!same) ++np;
      panel[i] = np;
      order[i] = theta_col_rank(k[8], k[9], k[10]);
    }
    Z.finalize_panels(panel, order);
  }
  st1.opA = OPA_N;
  st1.opB = OPB_N;
  tasks_to_stage(raw1, Z, st1);
  finalize_stage(st1, Z, Lenv, vec);
  for (size_t i = 0; i < raw.size(); ++i) {
    raw[i].lhs = Z.find(Zall.keys[raw_z[i]]);
    if (raw[i].lhs < 0) throw std::runtime_error("two-site task list: intermediate block missing");
  }
  st2.opA = OPA_N;
  st2.opB = OPB_T;
  tasks_to_stage(raw, vec, st2);
  finalize_stage(st2, vec, Z, Renv);
}

void emit_heff1(const BlockTensor& Lenv, const BlockTensor& Renv, const BlockTensor& vec, const MpoSite& W,
                BlockTensor& X, Stage& st1, Stage& st2) {
  emit_left_contraction(Lenv, vec, W, 0, X, st1);
  std::vector<RawTask> raw;
  for (size_t x = 0; x < X.keys.size(); ++x) {
    const Key& xk = X.keys[x];  // a'(0,1) s'(2) c'(3,4) w'(5) c(6,7)
    const Sector ap = key_sector(xk, 0), cp = key_sector(xk, 3), c = key_sector(xk, 6);
    const int ri = Renv.find(key_env(cp, xk[5], c));
    const Key ok = key_site(ap, xk[2], cp);
    if (ri < 0 || vec.find(ok) < 0) continue;
    RawTask t;
    t.out = ok;
    t.order = Key{c.q, c.tj, xk[5], 0, 0, 0, 0, 0, 0, 0, 0, 0};
    t.lhs = (int)x;
    t.rhs = ri;
    t.alpha = 1.0;
    raw.push_back(t);
  }
  st2.opA = OPA_N;
  st2.opB = OPB_T;
  tasks_to_stage(raw, vec, st2);
  finalize_stage(st2, vec, X, Renv);
}

void emit_env_left(const BlockTensor& Lenv, const BlockTensor& A, const MpoSite& W, BlockTensor& X,
                   BlockTensor& out, Stage& st1, Stage& st2) {
  emit_left_contraction(Lenv, A, W, 0, X, st1);
  std::vector<RawTask> raw;
  std::vector<Shape> shapes;
  for (size_t x = 0; x < X.keys.size(); ++x) {
    const Key& xk = X.keys[x];
    const Sector ap = key_sector(xk, 0), cp = key_sector(xk, 3), c = key_sector(xk, 6);
    const int ai = A.find(key_site(ap, xk[2], cp));
    if (ai < 0) continue;
    RawTask t;
    t.out = key_env(cp, xk[5], c);
    t.order = Key{ap.q, ap.tj, xk[2], 0, 0, 0, 0, 0, 0, 0, 0, 0};
    t.lhs = ai;
    t.rhs = (int)x;
    t.alpha = 1.0;
    raw.push_back(t);
    shapes.push_back(Shape{A.cols[ai], X.cols[x]});
  }
  layout_from_tasks(raw, shapes, 5, out);
  st2.opA = OPA_H;
  st2.opB = OPB_N;
  tasks_to_stage(raw, out, st2);
  finalize_stage(st2, out, A, X);
}

void emit_env_right(const BlockTensor& Renv, const BlockTensor& A, const MpoSite& W, BlockTensor& Y,
                    BlockTensor& out, Stage& st1, Stage& st2) {
  std::map<Sector, std::vector<int>> r_by_bp, a_by_b;
  for (size_t i = 0; i < Renv.keys.size(); ++i) r_by_bp[key_sector(Renv.keys[i], 0)].push_back((int)i);
  for (size_t i = 0; i < A.keys.size(); ++i) a_by_b[key_sector(A.keys[i], 3)].push_back((int)i);
  std::vector<RawTask> raw1, raw2;
  std::vector<Shape> shapes1, shapes2;
  std::map<Key, bool> ydone;
  struct Pending {
    Key ykey;
    RawTask t;
  };
  std::vector<Pending> pend;
  for (size_t ip = 0; ip < A.keys.size(); ++ip) {
    const Key& akp = A.keys[ip];  // c'(0,1) s'(2) b'(3,4)
    const Sector cp = key_sector(akp, 0), bp = key_sector(akp, 3);
    const int sp = akp[2];
    auto itr = r_by_bp.find(bp);
    if (itr == r_by_bp.end()) continue;
    for (int ri : itr->second) {
      const Key& rk = Renv.keys[ri];  // b'(0,1) w'(2) b(3,4)
      const int wp = rk[2];
      const Sector b = key_sector(rk, 3);
      const Key ykey{cp.q, cp.tj, sp, bp.q, bp.tj, wp, b.q, b.tj, 0, 0, 0, 0};
      auto ita = a_by_b.find(b);
      if (ita == a_by_b.end()) continue;
      for (int ai : ita->second) {
        const Key& ak = A.keys[ai];  // c(0,1) s(2) b(3,4)
        const Sector c = key_sector(ak, 0);
        const int s = ak[2];
        for (int w = 0; w < sym().nw; ++w) {
          const int tr = W.rank2[w][wp];
          if (tr < 0) continue;
          const double wv = W.val[w][wp][sp][s];
          if (wv == 0.0) continue;
          if (cp.q != c.q + MPO_Q[w] || !triangle(c.tj, MPO_TK[w], cp.tj)) continue;
          const double al = coef_right(c.tj, SITE_TJ[s], b.tj, MPO_TK[w], tr, MPO_TK[wp], cp.tj, SITE_TJ[sp], bp.tj) * wv;
          if (std::fabs(al) < ALPHA_ZERO) continue;
          if (!ydone.count(ykey)) {
            ydone[ykey] = true;
            RawTask t1;
            t1.out = ykey;
            t1.order = Key{0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
            t1.lhs = (int)ip;
            t1.rhs = ri;
            t1.alpha = 1.0;
            raw1.push_back(t1);
            shapes1.push_back(Shape{A.rows[ip], Renv.cols[ri]});
          }
          Pending p;
          p.ykey = ykey;
          p.t.out = key_env(cp, w, c);
          p.t.order = Key{sp, bp.q, bp.tj, wp, s, b.q, b.tj, 0, 0, 0, 0, 0};
          p.t.lhs = -1;
          p.t.rhs = ai;
          p.t.alpha = al;
          pend.push_back(p);
          shapes2.push_back(Shape{A.rows[ip], A.rows[ai]});
        }
      }
    }
  }
  layout_from_tasks(raw1, shapes1, 8, Y);
  st1.opA = OPA_C;
  st1.opB = OPB_N;
  tasks_to_stage(raw1, Y, st1);
  finalize_stage(st1, Y, A, Renv);
  for (auto& p : pend) {
    p.t.lhs = Y.find(p.ykey);
    raw2.push_back(p.t);
  }
  layout_from_tasks(raw2, shapes2, 5, out);
  st2.opA = OPA_N;
  st2.opB = OPB_T;
  tasks_to_stage(raw2, out, st2);
  finalize_stage(st2, out, Y, A);
}

void emit_merge(const BlockTensor& A1, const BlockTensor& A2, const BlockTensor& theta, Stage& st) {
  std::vector<RawTask> raw;
  for (size_t i = 0; i < theta.keys.size(); ++i) {
    const Key& k = theta.keys[i];
    const Sector a = key_sector(k, 0), c = key_sector(k, 3), b = key_sector(k, 6);
    const int i1 = A1.find(key_site(a, k[2], c)), i2 = A2.find(key_site(c, k[5], b));
    if (i1 < 0 || i2 < 0) continue;
    RawTask t;
    t.out = k;
    t.order = Key{0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    t.lhs = i1;
    t.rhs = i2;
    t.alpha = 1.0;
    t.scale = std::sqrt((double)(k[7] + 1));  // the two-site vector lives in the gauge sqrt(2 j_b + 1) theta
    raw.push_back(t);
  }
  st.opA = OPA_N;
  st.opB = OPB_N;
  tasks_to_stage(raw, theta, st);
  finalize_stage(st, theta, A1, A2);
}

void emit_heff0(const BlockTensor& Lenv, const BlockTensor& Renv, const BlockTensor& vec, BlockTensor& X,
                Stage& st1, Stage& st2) {
  std::vector<RawTask> raw1, raw2;
  std::vector<Shape> shapes1;
  struct Pend {
    Key xkey;
    RawTask t;
  };
  std::vector<Pend> pend;
  for (size_t e = 0; e < Lenv.keys.size(); ++e) {
    const Key& ek = Lenv.keys[e];  // c'(0,1) w(2) c(3,4)
    const Sector cp = key_sector(ek, 0), c = key_sector(ek, 3);
    const int ci = vec.find(Key{c.q, c.tj, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0});
    const int cpi = vec.find(Key{cp.q, cp.tj, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0});
    const int ri = Renv.find(ek);
    if (ci < 0 || cpi < 0 || ri < 0) continue;
    RawTask t1;
    t1.out = ek;
    t1.order = Key{0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    t1.lhs = (int)e;
    t1.rhs = ci;
    t1.alpha = 1.0;
    raw1.push_back(t1);
    shapes1.push_back(Shape{Lenv.rows[e], vec.cols[ci]});
    Pend p;
    p.xkey = ek;
    p.t.out = vec.keys[cpi];
    p.t.order = Key{c.q, c.tj, ek[2], 0, 0, 0, 0, 0, 0, 0, 0, 0};
    p.t.lhs = -1;
    p.t.rhs = ri;
    p.t.alpha = 1.0;
    pend.push_back(p);
  }
  layout_from_tasks(raw1, shapes1, 5, X);
  st1.opA = OPA_N;
  st1.opB = OPB_N;
  tasks_to_stage(raw1, X, st1);
  finalize_stage(st1, X, Lenv, vec);
  for (auto& p : pend) {
    p.t.lhs = X.find(p.xkey);
    raw2.push_back(p.t);
  }
  st2.opA = OPA_N;
  st2.opB = OPB_T;
  tasks_to_stage(raw2, vec, st2);
  finalize_stage(st2, vec, X, Renv);
}

void emit_absorb(const BlockTensor& C, const BlockTensor& A, const BlockTensor& Anew, bool left, Stage& st) {
  std::vector<RawTask> raw;
  for (size_t i = 0; i < Anew.keys.size(); ++i) {
    const Key& k = Anew.keys[i];  // x(0,1) s(2) y(3,4)
    const int ai = A.find(k);
    const Sector sec = left ? key_sector(k, 0) : key_sector(k, 3);
    const int ci = C.find(Key{sec.q, sec.tj, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0});
    if (ai < 0 || ci < 0) continue;
    RawTask t;
    t.out = k;
    t.order = Key{0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    t.lhs = left ? ci : ai;
    t.rhs = left ? ai : ci;
    t.alpha = 1.0;
    raw.push_back(t);
  }
  st.opA = OPA_N;
  st.opB = OPB_N;
  tasks_to_stage(raw, Anew, st);
  if (left) finalize_stage(st, Anew, C, A);
  else finalize_stage(st, Anew, A, C);
}

void emit_norm_env(const BlockTensor& Nenv, const BlockTensor& A, BlockTensor& Nout, Stage& st1, Stage& st2) {
  // stage 1: X[a,s,c] = N[a] A[a,s,c]  (X has A's layout);  stage 2: N'[c] = sum_{a,s} A[a,s,c]^H X[a,s,c]
  std::vector<RawTask> raw1, raw2;
  std::vector<Shape> shapes2;
  for (size_t i = 0; i < A.keys.size(); ++i) {
    const Key& k = A.keys[i];
    const Sector a = key_sector(k, 0), c = key_sector(k, 3);
    const int ni = Nenv.find(Key{a.q, a.tj, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0});
    if (ni < 0) continue;
    RawTask t;
    t.out = k;
    t.order = Key{0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    t.lhs = ni;
    t.rhs = (int)i;
    t.alpha = 1.0;
    raw1.push_back(t);
    RawTask u;
    u.out = Key{c.q, c.tj, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    u.order = Key{a.q, a.tj, k[2], 0, 0, 0, 0, 0, 0, 0, 0, 0};
    u.lhs = (int)i;
    u.rhs = (int)i;
    u.alpha = 1.0;
    raw2.push_back(u);
    shapes2.push_back(Shape{A.cols[i], A.cols[i]});
  }
  st1.opA = OPA_N;
  st1.opB = OPB_N;
  tasks_to_stage(raw1, A, st1);
  finalize_stage(st1, A, Nenv, A);
  layout_from_tasks(raw2, shapes2, 2, Nout);
  st2.opA = OPA_H;
  st2.opB = OPB_N;
  tasks_to_stage(raw2, Nout, st2);
  finalize_stage(st2, Nout, A, A);  // rhs = X which has A's layout
}

}  // namespace fh
