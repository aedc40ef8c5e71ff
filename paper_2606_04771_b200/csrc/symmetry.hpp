// Host symmetry layer: sector tables, block layouts, reduced MPO and task-list emission (H0).
#pragma once
#include "fh_internal.hpp"

namespace fh {

static const double ALPHA_ZERO = 1e-12;  // |alpha| below this counts as exactly 0 (reading A-14)

inline Key key_site(Sector a, int s, Sector c) { return Key{a.q, a.tj, s, c.q, c.tj, 0, 0, 0, 0, 0, 0, 0}; }
inline Key key_theta(Sector a, int s1, Sector c, int s2, Sector b) {
  return Key{a.q, a.tj, s1, c.q, c.tj, s2, b.q, b.tj, 0, 0, 0, 0};
}
inline Key key_env(Sector xp, int w, Sector x) { return Key{xp.q, xp.tj, w, x.q, x.tj, 0, 0, 0, 0, 0, 0, 0}; }

// all fusion-allowed one-site blocks (a,s,c) between two bonds
void layout_site(const Bond& bl, const Bond& br, BlockTensor& out);
// all fusion-allowed two-site blocks (a,s1,c,s2,b); c is any label allowed by fusion
void layout_theta(const Bond& bl, const Bond& br, BlockTensor& out);

void mpo_site_table(int site, double t_h, double U, MpoSite& out);

// Task lists.  Each emitter fills the intermediate tensor layout (Z / X / Y), the output layout
// where it is not given, and the two stages (host task arrays + GemmOut/GemmSeg + warp-unit list).
// two-site apply (H1 + H2): vec = theta layout (input and output)
void emit_heff2(const BlockTensor& Lenv, const BlockTensor& Renv, const BlockTensor& vec, const MpoSite& W1,
                const MpoSite& W2, BlockTensor& Z, Stage& st1, Stage& st2);
// one-site apply (H3): vec = site layout
void emit_heff1(const BlockTensor& Lenv, const BlockTensor& Renv, const BlockTensor& vec, const MpoSite& W,
                BlockTensor& X, Stage& st1, Stage& st2);
// left environment update (H4): out = new L layout (only blocks that receive a contribution)
void emit_env_left(const BlockTensor& Lenv, const BlockTensor& A, const MpoSite& W, BlockTensor& X,
                   BlockTensor& out, Stage& st1, Stage& st2);
// right environment update (H5)
void emit_env_right(const BlockTensor& Renv, const BlockTensor& A, const MpoSite& W, BlockTensor& Y,
                    BlockTensor& out, Stage& st1, Stage& st2);
// merge theta[a,s1,c,s2,b] = A1[a,s1,c] A2[c,s2,b] (H8): out = theta layout (given)
void emit_merge(const BlockTensor& A1, const BlockTensor& A2, const BlockTensor& theta, Stage& st);
// norm environment for measure_local (H10): X[a,s,c] = N[a] A[a,s,c];  N'[c] = sum_{a,s} A[a,s,c]^H X[a,s,c]
// N layouts use key {q, tj}.
void emit_norm_env(const BlockTensor& Nenv, const BlockTensor& A, BlockTensor& Nout, Stage& st1, Stage& st2);

// zero-site apply on a bond matrix C[c] (rows: bra-side dims, cols: ket-side dims), the backward step of
// one-site TDVP (NEXT-1): X[c',w,c] = L[c',w,c] C[c];  out[c'] = sum_{(c,w)} X[c',w,c] R[c',w,c]^T, coefficient 1
// (CG orthogonality).  vec = layout of C with keys {q, tj}.
void emit_heff0(const BlockTensor& Lenv, const BlockTensor& Renv, const BlockTensor& vec, BlockTensor& X,
                Stage& st1, Stage& st2);
// A'[c,s,b] = C[c] A[c,s,b] (left = true) or A'[a,s,c] = A[a,s,c] C[c] (left = false); Anew = layout of A'
void emit_absorb(const BlockTensor& C, const BlockTensor& A, const BlockTensor& Anew, bool left, Stage& st);

// fills outs/segs from the (sorted) task arrays and builds the warp-unit list
void finalize_stage(Stage& st, const BlockTensor& out, const BlockTensor& lhs, const BlockTensor& rhs);

}  // namespace fh
