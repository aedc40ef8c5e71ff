// Two-site TDVP sweep: merge (H8), Lanczos exponential (H6/H7 in api.cu),
// block-wise SVD + truncation (H9, vendor cuSOLVER, timed separately), environment update,
// one-site backward step (H3); and measure_local through norm environments (H10).
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <thread>

#include "context.hpp"

using namespace fh;

#define FH_CUSOLVER(x)                                                                    \
  do {                                                                                    \
    cusolverStatus_t st__ = (x);                                                          \
    if (st__ != CUSOLVER_STATUS_SUCCESS)                                                  \
      throw fh::FhError(FH_ECUDA, std::string(#x) + " failed, status " + std::to_string((int)st__)); \
  } while (0)

namespace {

// element (j, x) of a strided matrix is multiplied by s[j]
__global__ void scale_by_s_kernel(cplx* buf, int nj, int nx, int64_t stride_j, int64_t stride_x,
                                  const double* __restrict__ s) {
  const int64_t total = (int64_t)nj * nx;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int j = (int)(i / nx), x = (int)(i % nx);
    cplx* p = buf + j * stride_j + x * stride_x;
    const double f = s[j];
    p->x *= f;
    p->y *= f;
  }
}

struct SectorSvd {
  Sector c;
  int nrow, ncol, k;       // M_c is nrow x ncol, k = min
  bool transposed;         // buffer holds M_c^T row-major (== column-major M_c)
  int64_t m_off, u_off, vt_off, s_off;  // offsets into the scratch (complex / double units)
  std::vector<std::pair<Key, std::pair<int, int>>> rows;  // (a,s1) part: key{a.q,a.tj,s1}, (offset, dim)
  std::vector<std::pair<Key, std::pair<int, int>>> cols;  // (s2,b) part: key{s2,b.q,b.tj}
  int keep = 0;
  bool gram = false;       // factorised by the Gram-matrix eigenvalue route (svd_one): checked after the truncation
  // QR mode (one-site split): column-major A (qm x qn) at m_off, tau at u_off, R written to r_dst
  int qm = 0, qn = 0, r_ld = 0, r_transpose = 0;
  cplx* r_dst = nullptr;
};

// R factor out of the geqrf result (column-major A, ld m, upper trapezoid k x n): dst[j][x] = R[j][x]
// (row-major, ld) or, transposed, dst[x][j] = R[j][x]; the reflectors below the diagonal read as zero
__global__ void extract_r_kernel(const cplx* __restrict__ A, int m, int k, int n, cplx* __restrict__ dst, int ld,
                                 int transpose) {
  const int64_t total = (int64_t)k * n;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int j = (int)(i % k), x = (int)(i / k);
    const cplx v = j <= x ? A[j + (int64_t)x * m] : make_double2(0.0, 0.0);
    if (transpose) dst[(int64_t)x * ld + j] = v;
    else dst[(int64_t)j * ld + x] = v;
  }
}

// dst (n x n, column-major) = conj(src)^T
__global__ void conj_transpose_kernel(const cplx* __restrict__ src, cplx* __restrict__ dst, int n) {
  const int64_t total = (int64_t)n * n;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int r = (int)(i % n), c = (int)(i / n);  // dst(r, c) = conj(src(c, r))
    const cplx v = src[(int64_t)r * n + c];
    dst[i] = make_double2(v.x, -v.y);
  }
}

// ------------------------------------------------------------------------------------------
// Small sector matrices (G and V fit SMALL_SVD_SMEM, i.e. up to 82 x 82): one CTA of 8 to 32 warps per matrix, one launch for all of
// them -- one-sided (Hestenes) Jacobi SVD in shared memory.  B (m x n, m >= n, column-major) -> U (m x n),
// s (descending), V^H (n x n), the same conventions as cusolverDnZgesvd('S', 'S').  Column pairs (p, q) are
// rotated until every |g_p^H g_q| <= 1e-15 |g_p| |g_q|; the singular values are the final column norms
// (high relative accuracy, also for tiny ones).  At small chi a bond has tens of such matrices and a vendor
// call per matrix (0.25 ms each, host-blocking) dominated the sweep.
constexpr size_t SMALL_SVD_SMEM = 216 * 1024;
static inline size_t small_svd_bytes(int m, int n) {
  return ((size_t)m * n + (size_t)n * n) * sizeof(cplx) + (size_t)n * sizeof(double);
}
constexpr int FACT_NOT_CONVERGED = 1 << 20;  // status word of a Jacobi kernel that ran out of sweeps
constexpr int JACOBI_MAX_SWEEPS = 40;
struct SmallSvd {
  int64_t m_off, u_off, vt_off, s_off;
  int m, n;
  int stat, pad;  // index of the matrix' status word
};
__device__ __forceinline__ double warp_sum_all(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
constexpr int SMALL_SVD_MAX_WARPS = 32;  // the launch picks 8, 16 or 32 warps by the largest matrix of the batch
__global__ void __launch_bounds__(32 * SMALL_SVD_MAX_WARPS) small_svd_kernel(const SmallSvd* __restrict__ descs,
                                                                         cplx* __restrict__ buf,
                                                                         double* __restrict__ dS,
                                                                         int* __restrict__ status) {
  extern __shared__ __align__(16) unsigned char smem_svd[];
  __shared__ int rotated_any;
  bool converged = false;
  const SmallSvd d = descs[blockIdx.x];
  const int m = d.m, n = d.n, lane = threadIdx.x & 31, warp = threadIdx.x >> 5, tid = threadIdx.x;
  const int NT = blockDim.x, SMALL_SVD_WARPS = blockDim.x >> 5;
  cplx* G = reinterpret_cast<cplx*>(smem_svd);  // m x n column-major
  cplx* V = G + (size_t)m * n;                  // n x n column-major
  double* sig = reinterpret_cast<double*>(V + (size_t)n * n);
  const cplx* B = buf + d.m_off;
  for (int i = tid; i < m * n; i += NT) G[i] = B[i];
  for (int i = tid; i < n * n; i += NT) V[i] = make_double2((i % n) == (i / n) ? 1.0 : 0.0, 0.0);
  __syncthreads();
  // round-robin tournament: ne = n rounded up to even players, ne - 1 rounds of ne / 2 disjoint column pairs;
  // the pairs of a round are independent and go to different warps
  const int ne = (n + 1) & ~1;
  converged = n <= 1;
  for (int sweep = 0; sweep < JACOBI_MAX_SWEEPS && n > 1; ++sweep) {
    if (tid == 0) rotated_any = 0;
    __syncthreads();
    for (int r = 0; r < ne - 1; ++r) {
      for (int k = warp; k < ne / 2; k += SMALL_SVD_WARPS) {
        int p = (r + k) % (ne - 1);
        int q = k == 0 ? ne - 1 : (r - k + ne - 1) % (ne - 1);
        if (p > q) { const int t_ = p; p = q; q = t_; }
        if (q >= n) continue;  // dummy player of an odd n
        double a = 0.0, b = 0.0, cr = 0.0, ci = 0.0;
        for (int i = lane; i < m; i += 32) {
          const cplx x = G[p * m + i], y = G[q * m + i];
          a += x.x * x.x + x.y * x.y;
          b += y.x * y.x + y.y * y.y;
          cr += x.x * y.x + x.y * y.y;  // conj(x) * y
          ci += x.x * y.y - x.y * y.x;
        }
        a = warp_sum_all(a);
        b = warp_sum_all(b);
        cr = warp_sum_all(cr);
        ci = warp_sum_all(ci);
        const double c2 = cr * cr + ci * ci;
        if (c2 <= 1e-30 * a * b || c2 == 0.0) continue;
        if (lane == 0) rotated_any = 1;
        const double cabs = sqrt(c2);
        const double pr = cr / cabs, pi = ci / cabs;  // phase of c
        const double zeta = (b - a) / (2.0 * cabs);
        const double t = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
        const double cs = 1.0 / sqrt(1.0 + t * t), sn = cs * t;
        // y~ = conj(phase) * y;  x' = cs x - sn y~;  y' = sn x + cs y~
        for (int i = lane; i < m; i += 32) {
          const cplx x = G[p * m + i], y = G[q * m + i];
          const double yr = pr * y.x + pi * y.y, yi = pr * y.y - pi * y.x;
          G[p * m + i] = make_double2(cs * x.x - sn * yr, cs * x.y - sn * yi);
          G[q * m + i] = make_double2(sn * x.x + cs * yr, sn * x.y + cs * yi);
        }
        for (int i = lane; i < n; i += 32) {
          const cplx x = V[p * n + i], y = V[q * n + i];
          const double yr = pr * y.x + pi * y.y, yi = pr * y.y - pi * y.x;
          V[p * n + i] = make_double2(cs * x.x - sn * yr, cs * x.y - sn * yi);
          V[q * n + i] = make_double2(sn * x.x + cs * yr, sn * x.y + cs * yi);
        }
      }
      __syncthreads();
    }
    if (!rotated_any) {
      converged = true;
      break;
    }
    __syncthreads();
  }
  // singular values = column norms; rank by descending value (ties: lower column first)
  for (int j = warp; j < n; j += SMALL_SVD_WARPS) {
    double a = 0.0;
    for (int i = lane; i < m; i += 32) {
      const cplx x = G[j * m + i];
      a += x.x * x.x + x.y * x.y;
    }
    a = warp_sum_all(a);
    if (lane == 0) sig[j] = sqrt(a);
  }
  __syncthreads();
  if (tid == 0 && !converged) status[d.stat] = FACT_NOT_CONVERGED;
  cplx* U = buf + d.u_off;
  cplx* VT = buf + d.vt_off;
  double* S = dS + d.s_off;
  for (int j = warp; j < n; j += SMALL_SVD_WARPS) {
    const double sj = sig[j];
    int rank = 0;
    for (int l = 0; l < n; ++l) rank += (sig[l] > sj || (sig[l] == sj && l < j)) ? 1 : 0;
    const double inv = sj > 0.0 ? 1.0 / sj : 0.0;
    if (lane == 0) S[rank] = sj;
    for (int i = lane; i < m; i += 32) {
      const cplx x = G[j * m + i];
      U[(size_t)rank * m + i] = make_double2(x.x * inv, x.y * inv);
    }
    for (int i = lane; i < n; i += 32) {  // V^H[rank][i] = conj(V[i][j]), column-major n x n
      const cplx x = V[j * n + i];
      VT[(size_t)i * n + rank] = make_double2(x.x, -x.y);
    }
  }
}

// ------------------------------------------------------------------------------------------
// Mid-size sector matrices (too large for small_svd_kernel, n <= 128 by default, FH_SVD_MID_MAXN): the same one-sided Jacobi, one
// 32-warp CTA per matrix, working IN PLACE on B in global memory with V in arena scratch.  A matrix of this size
// (B and V together 0.3-0.7 MB) stays in the L1/L2 of its SM, and all accesses of a column pair come from one
// warp, with __syncthreads between tournament rounds, so plain loads and stores are coherent.  It is slower per
// matrix than the vendor routine (about 10 ms against 5 ms) but it is ONE launch for all of them on a side
// stream, while the vendor drivers, which are bound by their ~800 launches per matrix on the host threads, work
// through the larger matrices: every matrix moved here shortens the vendor queue of the bond.
struct MidSvd {
  int64_t m_off, u_off, vt_off, s_off, v_off;  // v_off relative to the V scratch base
  int m, n;
  int stat, pad;
};
constexpr int MID_SVD_HARD_MAXN = 256;
__global__ void __launch_bounds__(1024) mid_svd_kernel(const MidSvd* __restrict__ descs, cplx* buf, cplx* vbase,
                                                       double* __restrict__ dS, int* __restrict__ status) {
  __shared__ int rotated_any;
  bool converged = false;
  __shared__ double sig[MID_SVD_HARD_MAXN];
  const MidSvd d = descs[blockIdx.x];
  const int m = d.m, n = d.n, lane = threadIdx.x & 31, warp = threadIdx.x >> 5, tid = threadIdx.x;
  const int NT = blockDim.x, NW = blockDim.x >> 5;
  cplx* G = buf + d.m_off;   // m x n column-major, rotated in place
  cplx* V = vbase + d.v_off;  // n x n column-major
  for (int i = tid; i < n * n; i += NT) V[i] = make_double2((i % n) == (i / n) ? 1.0 : 0.0, 0.0);
  __syncthreads();
  const int ne = (n + 1) & ~1;
  converged = n <= 1;
  for (int sweep = 0; sweep < JACOBI_MAX_SWEEPS && n > 1; ++sweep) {
    if (tid == 0) rotated_any = 0;
    __syncthreads();
    for (int r = 0; r < ne - 1; ++r) {
      for (int k = warp; k < ne / 2; k += NW) {
        int p = (r + k) % (ne - 1);
        int q = k == 0 ? ne - 1 : (r - k + ne - 1) % (ne - 1);
        if (p > q) { const int t_ = p; p = q; q = t_; }
        if (q >= n) continue;
        cplx* gp = G + (size_t)p * m;
        cplx* gq = G + (size_t)q * m;
        double a = 0.0, b = 0.0, cr = 0.0, ci = 0.0;
        for (int i = lane; i < m; i += 32) {
          const cplx x = gp[i], y = gq[i];
          a += x.x * x.x + x.y * x.y;
          b += y.x * y.x + y.y * y.y;
          cr += x.x * y.x + x.y * y.y;
          ci += x.x * y.y - x.y * y.x;
        }
        a = warp_sum_all(a);
        b = warp_sum_all(b);
        cr = warp_sum_all(cr);
        ci = warp_sum_all(ci);
        const double c2 = cr * cr + ci * ci;
        if (c2 <= 1e-30 * a * b || c2 == 0.0) continue;
        if (lane == 0) rotated_any = 1;
        const double cabs = sqrt(c2);
        const double pr = cr / cabs, pi = ci / cabs;
        const double zeta = (b - a) / (2.0 * cabs);
        const double t = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
        const double cs = 1.0 / sqrt(1.0 + t * t), sn = cs * t;
        for (int i = lane; i < m; i += 32) {
          const cplx x = gp[i], y = gq[i];
          const double yr = pr * y.x + pi * y.y, yi = pr * y.y - pi * y.x;
          gp[i] = make_double2(cs * x.x - sn * yr, cs * x.y - sn * yi);
          gq[i] = make_double2(sn * x.x + cs * yr, sn * x.y + cs * yi);
        }
        cplx* vp = V + (size_t)p * n;
        cplx* vq = V + (size_t)q * n;
        for (int i = lane; i < n; i += 32) {
          const cplx x = vp[i], y = vq[i];
          const double yr = pr * y.x + pi * y.y, yi = pr * y.y - pi * y.x;
          vp[i] = make_double2(cs * x.x - sn * yr, cs * x.y - sn * yi);
          vq[i] = make_double2(sn * x.x + cs * yr, sn * x.y + cs * yi);
        }
      }
      __syncthreads();
    }
    if (!rotated_any) {
      converged = true;
      break;
    }
    __syncthreads();
  }
  for (int j = warp; j < n; j += NW) {
    double a = 0.0;
    for (int i = lane; i < m; i += 32) {
      const cplx x = G[(size_t)j * m + i];
      a += x.x * x.x + x.y * x.y;
    }
    a = warp_sum_all(a);
    if (lane == 0) sig[j] = sqrt(a);
  }
  __syncthreads();
  if (tid == 0 && !converged) status[d.stat] = FACT_NOT_CONVERGED;
  cplx* U = buf + d.u_off;
  cplx* VT = buf + d.vt_off;
  double* S = dS + d.s_off;
  for (int j = warp; j < n; j += NW) {
    const double sj = sig[j];
    int rank = 0;
    for (int l = 0; l < n; ++l) rank += (sig[l] > sj || (sig[l] == sj && l < j)) ? 1 : 0;
    const double inv = sj > 0.0 ? 1.0 / sj : 0.0;
    if (lane == 0) S[rank] = sj;
    for (int i = lane; i < m; i += 32) {
      const cplx x = G[(size_t)j * m + i];
      U[(size_t)rank * m + i] = make_double2(x.x * inv, x.y * inv);
    }
    for (int i = lane; i < n; i += 32) {
      const cplx x = V[(size_t)j * n + i];
      VT[(size_t)i * n + rank] = make_double2(x.x, -x.y);
    }
  }
}

// ------------------------------------------------------------------------------------------
// Small one-site splits (the whole qm x qn sector matrix fits shared memory): Householder QR in one launch for
// all of them, one CTA of 8 to 32 warps per matrix.  Same conventions as cusolverDnZgeqrf + Zungqr (LAPACK zlarfg /
// zung2r: H_j = I - tau_j v v^H with v_0 = 1, real diagonal of R): column-major A (m x n) at m_off is
// replaced by Q (m x k, k = min(m, n)), R (k x n) goes straight to r_dst like extract_r_kernel writes it.
struct SmallQr {
  int64_t m_off;
  cplx* r_dst;
  int m, n, r_ld, r_transpose;
};
constexpr size_t SMALL_QR_SMEM = 180 * 1024;
constexpr int SMALL_QR_MAX_WARPS = 32;  // the launch picks 8, 16 or 32 warps by the widest matrix of the batch
constexpr int SMALL_QR_MAXK = 256;
__global__ void __launch_bounds__(32 * SMALL_QR_MAX_WARPS) small_qr_kernel(const SmallQr* __restrict__ descs,
                                                                       cplx* __restrict__ buf) {
  extern __shared__ __align__(16) unsigned char smem_qr[];
  __shared__ cplx tau_s[SMALL_QR_MAXK];
  const SmallQr d = descs[blockIdx.x];
  const int m = d.m, n = d.n, k = min(m, n);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, tid = threadIdx.x;
  const int NT = blockDim.x, SMALL_QR_WARPS = blockDim.x >> 5;
  cplx* A = reinterpret_cast<cplx*>(smem_qr);  // m x n column-major
  cplx* Ag = buf + d.m_off;
  for (int i = tid; i < m * n; i += NT) A[i] = Ag[i];
  __syncthreads();
  // ---- factorisation: H_j^H ... H_0^H A = R
  for (int j = 0; j < k; ++j) {
    cplx* x = A + (size_t)j * m;
    if (warp == 0) {  // zlarfg on x[j..m)
      double xn2 = 0.0;
      for (int i = j + 1 + lane; i < m; i += 32) xn2 += x[i].x * x[i].x + x[i].y * x[i].y;
      xn2 = warp_sum_all(xn2);
      const cplx alpha = x[j];
      cplx tau = make_double2(0.0, 0.0);
      if (xn2 > 0.0 || alpha.y != 0.0) {
        const double nrm = sqrt(alpha.x * alpha.x + alpha.y * alpha.y + xn2);
        const double beta = alpha.x >= 0.0 ? -nrm : nrm;
        tau = make_double2((beta - alpha.x) / beta, -alpha.y / beta);
        // v[i] = x[i] / (alpha - beta)
        const double dr = alpha.x - beta, di = alpha.y, dd = dr * dr + di * di;
        const double ir = dr / dd, ii = -di / dd;
        for (int i = j + 1 + lane; i < m; i += 32) {
          const cplx v = x[i];
          x[i] = make_double2(v.x * ir - v.y * ii, v.x * ii + v.y * ir);
        }
        __syncwarp();
        if (lane == 0) x[j] = make_double2(beta, 0.0);
      }
      if (lane == 0) tau_s[j] = tau;
    }
    __syncthreads();
    const cplx tau = tau_s[j];
    if (tau.x != 0.0 || tau.y != 0.0) {
      // apply H_j^H = I - conj(tau) v v^H to the trailing columns, one warp per column
      for (int c = j + 1 + warp; c < n; c += SMALL_QR_WARPS) {
        cplx* y = A + (size_t)c * m;
        double wr = 0.0, wi = 0.0;  // w = v^H y, v_j = 1
        for (int i = j + 1 + lane; i < m; i += 32) {
          const cplx v = x[i], yy = y[i];
          wr += v.x * yy.x + v.y * yy.y;
          wi += v.x * yy.y - v.y * yy.x;
        }
        wr = warp_sum_all(wr);
        wi = warp_sum_all(wi);
        wr += y[j].x;
        wi += y[j].y;
        const double fr = tau.x * wr + tau.y * wi, fi = tau.x * wi - tau.y * wr;  // conj(tau) * w
        for (int i = j + 1 + lane; i < m; i += 32) {
          const cplx v = x[i];
          y[i].x -= fr * v.x - fi * v.y;
          y[i].y -= fr * v.y + fi * v.x;
        }
        __syncwarp();
        if (lane == 0) {
          y[j].x -= fr;
          y[j].y -= fi;
        }
      }
    }
    __syncthreads();
  }
  // ---- R out (upper trapezoid k x n; zeros below the diagonal)
  for (int i = tid; i < k * n; i += NT) {
    const int r = i % k, c = i / k;
    const cplx v = r <= c ? A[(size_t)c * m + r] : make_double2(0.0, 0.0);
    if (d.r_transpose) d.r_dst[(int64_t)c * d.r_ld + r] = v;
    else d.r_dst[(int64_t)r * d.r_ld + c] = v;
  }
  __syncthreads();
  // ---- Q = H_0 ... H_{k-1} (first k columns), in place (zung2r)
  for (int j = k - 1; j >= 0; --j) {
    cplx* x = A + (size_t)j * m;
    const cplx tau = tau_s[j];
    if (tau.x != 0.0 || tau.y != 0.0) {
      for (int c = j + 1 + warp; c < k; c += SMALL_QR_WARPS) {  // apply H_j = I - tau v v^H from the left
        cplx* y = A + (size_t)c * m;
        double wr = 0.0, wi = 0.0;
        for (int i = j + 1 + lane; i < m; i += 32) {
          const cplx v = x[i], yy = y[i];
          wr += v.x * yy.x + v.y * yy.y;
          wi += v.x * yy.y - v.y * yy.x;
        }
        wr = warp_sum_all(wr);
        wi = warp_sum_all(wi);
        wr += y[j].x;
        wi += y[j].y;
        const double fr = tau.x * wr - tau.y * wi, fi = tau.x * wi + tau.y * wr;  // tau * w
        for (int i = j + 1 + lane; i < m; i += 32) {
          const cplx v = x[i];
          y[i].x -= fr * v.x - fi * v.y;
          y[i].y -= fr * v.y + fi * v.x;
        }
        __syncwarp();
        if (lane == 0) {
          y[j].x -= fr;
          y[j].y -= fi;
        }
      }
    }
    __syncthreads();
    // column j itself: -tau v below the diagonal, 1 - tau on it, zeros above
    for (int i = tid; i < m; i += NT) {
      cplx v;
      if (i < j) v = make_double2(0.0, 0.0);
      else if (i == j) v = make_double2(1.0 - tau.x, -tau.y);
      else v = make_double2(-(tau.x * x[i].x - tau.y * x[i].y), -(tau.x * x[i].y + tau.y * x[i].x));
      x[i] = v;
    }
    __syncthreads();
  }
  for (int i = tid; i < m * k; i += NT) Ag[i] = A[i];
}

void worker_reserve(fh_ctx::SvdWorker& w, size_t bytes) {
  if (bytes <= w.dwork_bytes) return;
  bytes = std::max<size_t>(bytes, (size_t)48 << 20);  // at least 48 MB: covers chi = 4096 without growing again
  FH_CUDA(cudaStreamSynchronize(w.s));
  if (w.dwork) FH_CUDA(cudaFree(w.dwork));
  w.dwork = nullptr;
  w.dwork_bytes = bytes + bytes / 2;
  FH_CUDA(cudaMalloc(&w.dwork, w.dwork_bytes));
}

// Gram-matrix eigenvalue route, last step: eigenpairs of G = B^H B (ascending, vectors in the columns of W) ->
// singular values (descending), V^H (n x n, ld n) and Vs = V Sigma^-1 (n x n, ld n; zero columns where sigma = 0)
__global__ void gram_finish_kernel(const cplx* __restrict__ W, const double* __restrict__ lam, int n, double* __restrict__ sv,
                                   cplx* __restrict__ VT, cplx* __restrict__ Vs) {
  const int64_t total = (int64_t)n * n;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
    const int j = (int)(e % n), i = (int)(e / n);  // component j of right singular vector i
    const double l = lam[n - 1 - i];
    const double sg = l > 0.0 ? sqrt(l) : 0.0;
    const cplx v = W[j + (int64_t)(n - 1 - i) * n];
    VT[i + (int64_t)j * n] = make_double2(v.x, -v.y);
    const double r = sg > 0.0 ? 1.0 / sg : 0.0;
    Vs[j + (int64_t)i * n] = make_double2(v.x * r, v.y * r);
    if (j == 0) sv[i] = sg;
  }
}

// Batched form of the Gram route (gram_batch below): the Gram matrix of a sector sits in the top-left n x n block of
// an npad x npad slot (ld npad); this kernel, launched after the ZGEMM that wrote the block, clears the rest of the
// slot and puts -(1 + trace G) on the padded diagonal: npad - n eigenvalues below every true one (>= 0), whose
// eigenvectors are unit vectors of the padding, so the true eigenpairs are the LAST n of the ascending list.
__global__ void gram_pad_kernel(cplx* __restrict__ G, int n, int npad) {
  __shared__ double tr;
  if (threadIdx.x < 32) {
    double t = 0.0;
    for (int i = threadIdx.x; i < n; i += 32) t += G[i + (int64_t)i * npad].x;
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (threadIdx.x == 0) tr = t;
  }
  __syncthreads();
  const double pad = -(1.0 + tr);
  const int64_t total = (int64_t)npad * npad;
  for (int64_t e = threadIdx.x; e < total; e += blockDim.x) {
    const int i = (int)(e % npad), j = (int)(e / npad);
    if (i >= n || j >= n) G[e] = make_double2(i == j ? pad : 0.0, 0.0);
  }
}
// as gram_finish_kernel, eigenpairs taken from an npad-wide slot (W: ld npad, lam: npad values, the last n are the sector's)
__global__ void gram_finish_padded_kernel(const cplx* __restrict__ W, const double* __restrict__ lam, int n, int npad,
                                          double* __restrict__ sv, cplx* __restrict__ VT, cplx* __restrict__ Vs) {
  const int64_t total = (int64_t)n * n;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
    const int j = (int)(e % n), i = (int)(e / n);
    const double l = lam[npad - 1 - i];
    const double sg = l > 0.0 ? sqrt(l) : 0.0;
    const cplx v = W[j + (int64_t)(npad - 1 - i) * npad];
    VT[i + (int64_t)j * n] = make_double2(v.x, -v.y);
    const double r = sg > 0.0 ? 1.0 / sg : 0.0;
    Vs[j + (int64_t)i * n] = make_double2(v.x * r, v.y * r);
    if (j == 0) sv[i] = sg;
  }
}

const int GESVDP_MIN_N = 48;  // below this the QR-iteration driver is as fast and has no conditioning caveat

// SVD of one sector matrix on worker w: column-major B (m x n, m >= n) at buf + m_off ->
// s (n), U (m x n, ld m) at u_off, V^H (n x n, ld n) at vt_off.
// n >= GESVDP_MIN_N: cusolverDnXgesvdp (polar decomposition + Hermitian eigensolver; measured 3.3x
// faster than Zgesvd at n = 600) on a copy; if it reports a perturbation of the spectrum
// (err_sigma != 0: numerically rank-deficient input) the QR-iteration driver Zgesvd redoes it.
//
// Gram route (gram_minn > 0 and n >= gram_minn): G = B^H B (one ZGEMM), Hermitian eigendecomposition G = V Lambda V^H
// (cusolverDnZheevd: 8 ms at n = 600 where gesvdp takes 23 ms, and the largest sector matrix of a bond is the
// critical path of the whole SVD phase: the phase does not depend on the number of workers), sigma = sqrt(lambda),
// U = B V Sigma^-1 (one ZGEMM).  Squaring the matrix costs accuracy for SMALL singular values only: sigma_i comes out
// with an absolute error of eps sigma_max^2 / (2 sigma_i) and the columns of U are orthonormal to eps (sigma_max /
// sigma_i)^2.  The caller therefore accepts the result of a sector only if every singular value the truncation KEEPS
// is >= GRAM_SAFE_RATIO sigma_max of that sector, and sends the sector through the routes below otherwise
// (svd_split).  In a chi-capped sweep the kept values of the large sectors are >= 1e-2 sigma_max.
const double GRAM_SAFE_RATIO = 3e-3;  // U orthonormal to 1.2e-11, sigma to 2e-14 sigma_max
void svd_one(fh_ctx::SvdWorker& w, SectorSvd& S, cplx* buf, double* dS, int64_t* counts, int* d_status, int gram_minn) {
  const int m = std::max(S.nrow, S.ncol), n = S.k;
  cuDoubleComplex* A = (cuDoubleComplex*)(buf + S.m_off);
  cuDoubleComplex* U = (cuDoubleComplex*)(buf + S.u_off);
  cuDoubleComplex* VT = (cuDoubleComplex*)(buf + S.vt_off);
  double* sv = dS + S.s_off;
  S.gram = false;
  if (gram_minn > 0 && n >= gram_minn) {
    const size_t g_bytes = ((size_t)n * n * sizeof(cplx) + 255) / 256 * 256;
    const size_t l_bytes = ((size_t)n * sizeof(double) + 255) / 256 * 256;
    int lwork = 0;
    FH_CUSOLVER(cusolverDnZheevd_bufferSize(w.h, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, n, nullptr, n, nullptr, &lwork));
    worker_reserve(w, 2 * g_bytes + l_bytes + (size_t)lwork * sizeof(cuDoubleComplex) + 256);
    char* base = (char*)w.dwork;
    cuDoubleComplex* G = (cuDoubleComplex*)base;
    cuDoubleComplex* Vs = (cuDoubleComplex*)(base + g_bytes);
    double* lam = (double*)(base + 2 * g_bytes);
    cuDoubleComplex* work = (cuDoubleComplex*)(base + 2 * g_bytes + l_bytes);
    const cuDoubleComplex one = make_cuDoubleComplex(1.0, 0.0), zero = make_cuDoubleComplex(0.0, 0.0);
    FH_REQUIRE(cublasZgemm(w.cb, CUBLAS_OP_C, CUBLAS_OP_N, n, n, m, &one, A, m, A, m, &zero, G, n) == CUBLAS_STATUS_SUCCESS,
               FH_ECUDA, "svd: cublasZgemm (Gram matrix) failed");
    FH_CUSOLVER(cusolverDnZheevd(w.h, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, n, G, n, lam, work, lwork, w.d_info));
    const int64_t tot = (int64_t)n * n;
    gram_finish_kernel<<<(int)std::min<int64_t>((tot + 255) / 256, 1184), 256, 0, w.s>>>((const cplx*)G, lam, n, sv, (cplx*)VT,
                                                                                     (cplx*)Vs);
    FH_REQUIRE(cublasZgemm(w.cb, CUBLAS_OP_N, CUBLAS_OP_N, m, n, n, &one, A, m, Vs, n, &zero, U, m) == CUBLAS_STATUS_SUCCESS,
               FH_ECUDA, "svd: cublasZgemm (U = B V / sigma) failed");
    FH_CUDA(cudaMemcpyAsync(d_status, w.d_info, sizeof(int), cudaMemcpyDeviceToDevice, w.s));
    S.gram = true;
    ++counts[3];
    return;
  }
  if (n >= GESVDP_MIN_N) {
    const size_t a_bytes = ((size_t)m * n * sizeof(cplx) + 255) / 256 * 256;
    const size_t v_bytes = ((size_t)n * n * sizeof(cplx) + 255) / 256 * 256;
    size_t wd = 0, wh = 0;
    FH_CUSOLVER(cusolverDnXgesvdp_bufferSize(w.h, w.params, CUSOLVER_EIG_MODE_VECTOR, 1, m, n, CUDA_C_64F, A, m,
                                             CUDA_R_64F, sv, CUDA_C_64F, U, m, CUDA_C_64F, VT, n, CUDA_C_64F, &wd, &wh));
    worker_reserve(w, a_bytes + v_bytes + wd + 256);
    if (w.hwork.size() < wh + 16) w.hwork.resize(wh + 16);
    char* base = (char*)w.dwork;
    cuDoubleComplex* Ac = (cuDoubleComplex*)base;
    cuDoubleComplex* V = (cuDoubleComplex*)(base + a_bytes);
    void* ws = base + a_bytes + v_bytes;
    FH_CUDA(cudaMemcpyAsync(Ac, A, (size_t)m * n * sizeof(cplx), cudaMemcpyDeviceToDevice, w.s));
    double err_sigma = 0.0;
    FH_CUSOLVER(cusolverDnXgesvdp(w.h, w.params, CUSOLVER_EIG_MODE_VECTOR, 1, m, n, CUDA_C_64F, Ac, m, CUDA_R_64F, sv,
                                  CUDA_C_64F, U, m, CUDA_C_64F, V, n, CUDA_C_64F, ws, wd, w.hwork.data(), wh, w.d_info,
                                  &err_sigma));
    if (err_sigma == 0.0) {
      const int64_t tot = (int64_t)n * n;
      conj_transpose_kernel<<<(int)std::min<int64_t>((tot + 255) / 256, 1184), 256, 0, w.s>>>((const cplx*)V, (cplx*)VT, n);
      FH_CUDA(cudaMemcpyAsync(d_status, w.d_info, sizeof(int), cudaMemcpyDeviceToDevice, w.s));
      ++counts[1];
      return;
    }
    ++counts[2];
  }
  int lwork = 0;
  FH_CUSOLVER(cusolverDnZgesvd_bufferSize(w.h, m, n, &lwork));
  worker_reserve(w, (size_t)lwork * sizeof(cuDoubleComplex));
  FH_CUSOLVER(cusolverDnZgesvd(w.h, 'S', 'S', m, n, A, m, sv, U, m, VT, n, (cuDoubleComplex*)w.dwork,
                               (int)(w.dwork_bytes / sizeof(cuDoubleComplex)), nullptr, w.d_info));
  FH_CUDA(cudaMemcpyAsync(d_status, w.d_info, sizeof(int), cudaMemcpyDeviceToDevice, w.s));
  ++counts[0];
}

// The Gram route for SEVERAL sectors at once: their Gram matrices, padded to a common size, go through ONE
// cusolverDnXsyevBatched call.  Why: a vendor eigensolver is a chain of ~1500 small dependent kernels (4.3 ms alone at
// n = 352), and sixteen chains side by side take 20 ms per bond whatever the number of host threads -- the GPU front
// end is what they queue on; the batched solver walks ONE chain for all of them (1.7 / 9.5 / 19.7 ms for 16 matrices of
// 128 / 224 / 352 columns, measured), so the mid-sized majority is taken out of the queue of the few largest.
void gram_batch(fh_ctx::SvdWorker& w, const std::vector<SectorSvd*>& order, const std::vector<int>& gb, cplx* buf, double* dS,
                int* d_status) {
  const int nb = (int)gb.size();
  int npad = 0;
  for (int x : gb) npad = std::max(npad, order[x]->k);
  npad = (npad + 31) / 32 * 32;
  const size_t slot = (size_t)npad * npad;
  const size_t g_bytes = (slot * nb * sizeof(cplx) + 255) / 256 * 256;
  const size_t l_bytes = ((size_t)npad * nb * sizeof(double) + 255) / 256 * 256;
  const size_t i_bytes = ((size_t)nb * sizeof(int) + 255) / 256 * 256;
  size_t wd = 0, wh = 0;
  FH_CUSOLVER(cusolverDnXsyevBatched_bufferSize(w.h, w.params, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, npad, CUDA_C_64F,
                                                nullptr, npad, CUDA_R_64F, nullptr, CUDA_C_64F, &wd, &wh, nb));
  worker_reserve(w, 2 * g_bytes + l_bytes + i_bytes + wd + 256);
  if (w.hwork.size() < wh + 16) w.hwork.resize(wh + 16);
  char* base = (char*)w.dwork;
  cuDoubleComplex* G = (cuDoubleComplex*)base;
  cuDoubleComplex* Vs = (cuDoubleComplex*)(base + g_bytes);
  double* lam = (double*)(base + 2 * g_bytes);
  int* info = (int*)(base + 2 * g_bytes + l_bytes);
  void* ws = base + 2 * g_bytes + l_bytes + i_bytes;
  const cuDoubleComplex one = make_cuDoubleComplex(1.0, 0.0), zero = make_cuDoubleComplex(0.0, 0.0);
  for (int x = 0; x < nb; ++x) {
    const SectorSvd& S = *order[gb[x]];
    const int m = std::max(S.nrow, S.ncol), n = S.k;
    const cuDoubleComplex* A = (const cuDoubleComplex*)(buf + S.m_off);
    FH_REQUIRE(cublasZgemm(w.cb, CUBLAS_OP_C, CUBLAS_OP_N, n, n, m, &one, A, m, A, m, &zero, G + x * slot, npad) ==
                   CUBLAS_STATUS_SUCCESS,
               FH_ECUDA, "svd: cublasZgemm (Gram matrix, batched route) failed");
    gram_pad_kernel<<<1, 1024, 0, w.s>>>((cplx*)(G + x * slot), n, npad);
  }
  FH_CUSOLVER(cusolverDnXsyevBatched(w.h, w.params, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, npad, CUDA_C_64F, G, npad,
                                     CUDA_R_64F, lam, CUDA_C_64F, ws, wd, w.hwork.data(), wh, info, nb));
  for (int x = 0; x < nb; ++x) {
    SectorSvd& S = *order[gb[x]];
    const int m = std::max(S.nrow, S.ncol), n = S.k;
    const cuDoubleComplex* A = (const cuDoubleComplex*)(buf + S.m_off);
    const int64_t tot = (int64_t)n * n;
    gram_finish_padded_kernel<<<(int)std::min<int64_t>((tot + 255) / 256, 296), 256, 0, w.s>>>(
        (const cplx*)(G + x * slot), lam + (size_t)x * npad, n, npad, dS + S.s_off, buf + S.vt_off, (cplx*)(Vs + x * slot));
    FH_REQUIRE(cublasZgemm(w.cb, CUBLAS_OP_N, CUBLAS_OP_N, m, n, n, &one, A, m, Vs + x * slot, n, &zero,
                           (cuDoubleComplex*)(buf + S.u_off), m) == CUBLAS_STATUS_SUCCESS,
               FH_ECUDA, "svd: cublasZgemm (U = B V / sigma, batched route) failed");
    FH_CUDA(cudaMemcpyAsync(d_status + gb[x], info + x, sizeof(int), cudaMemcpyDeviceToDevice, w.s));
    S.gram = true;
  }
}

// Householder QR of one sector matrix (one-site split, no truncation): geqrf, R copied out, ungqr in place.
void qr_one(fh_ctx::SvdWorker& w, const SectorSvd& S, cplx* buf, int* d_status, int* d_status2) {
  const int m = S.qm, n = S.qn, k = std::min(m, n);
  cuDoubleComplex* A = (cuDoubleComplex*)(buf + S.m_off);
  cuDoubleComplex* tau = (cuDoubleComplex*)(buf + S.u_off);
  int lw1 = 0, lw2 = 0;
  FH_CUSOLVER(cusolverDnZgeqrf_bufferSize(w.h, m, n, A, m, &lw1));
  FH_CUSOLVER(cusolverDnZungqr_bufferSize(w.h, m, k, k, A, m, tau, &lw2));
  const int lwork = std::max(lw1, lw2);
  worker_reserve(w, (size_t)lwork * sizeof(cuDoubleComplex) + 256);
  FH_CUSOLVER(cusolverDnZgeqrf(w.h, m, n, A, m, tau, (cuDoubleComplex*)w.dwork, lwork, w.d_info));
  FH_CUDA(cudaMemcpyAsync(d_status, w.d_info, sizeof(int), cudaMemcpyDeviceToDevice, w.s));
  const int64_t tot = (int64_t)k * n;
  extract_r_kernel<<<(int)std::min<int64_t>((tot + 255) / 256, 1184), 256, 0, w.s>>>((const cplx*)A, m, k, n, S.r_dst, S.r_ld,
                                                                                     S.r_transpose);
  FH_CUSOLVER(cusolverDnZungqr(w.h, m, k, k, A, m, tau, (cuDoubleComplex*)w.dwork, lwork, w.d_info));
  FH_CUDA(cudaMemcpyAsync(d_status2, w.d_info, sizeof(int), cudaMemcpyDeviceToDevice, w.s));
}

// Descriptors of the small-matrix kernels go through a host buffer owned by the context (it outlives the
// asynchronous copy; the event guards its reuse), so their launch needs no stream synchronisation.
const void* stage_small_desc(fh_ctx* ctx, const void* src, size_t bytes) {
  if (ctx->small_copied_armed) FH_CUDA(cudaEventSynchronize(ctx->small_copied));
  ctx->small_copied_armed = true;
  if (ctx->small_desc_host.size() < bytes) ctx->small_desc_host.resize(bytes + bytes / 2);
  std::memcpy(ctx->small_desc_host.data(), src, bytes);
  return ctx->small_desc_host.data();
}

// All sector SVDs of one bond (H9), heaviest first, pulled by host worker threads from a shared
// counter; every worker has its own cuSOLVER handle, stream and workspace.  The main stream forks
// into the worker streams and joins them again through events, so the phase timers on the main
// stream cover the whole batch.
void run_sector_svds(fh_ctx* ctx, const std::vector<SectorSvd*>& order, cplx* buf, double* dS, bool qr = false,
                     bool allow_gram = true) {
  const int gram_minn = (allow_gram && !qr) ? ctx->opt_svd_gram_minn : 0;
  if (ctx->svd_workers.empty()) {
    int nw = (int)std::thread::hardware_concurrency() - 1;
    if (ctx->opt_svd_threads > 0) nw = ctx->opt_svd_threads;
    nw = std::max(1, std::min(nw, 12));
    ctx->svd_workers.resize(nw);
    for (auto& w : ctx->svd_workers) {
      FH_CUDA(cudaStreamCreateWithFlags(&w.s, cudaStreamNonBlocking));
      FH_CUSOLVER(cusolverDnCreate(&w.h));
      FH_CUSOLVER(cusolverDnSetStream(w.h, w.s));
      FH_CUSOLVER(cusolverDnCreateParams(&w.params));
      FH_REQUIRE(cublasCreate(&w.cb) == CUBLAS_STATUS_SUCCESS, FH_ECUDA, "cublasCreate failed");
      cublasSetStream(w.cb, w.s);
      FH_CUDA(cudaMalloc((void**)&w.d_info, sizeof(int)));
      FH_CUDA(cudaEventCreateWithFlags(&w.done, cudaEventDisableTiming));
    }
    FH_CUDA(cudaEventCreateWithFlags(&ctx->svd_fork, cudaEventDisableTiming));
    FH_CUDA(cudaEventCreateWithFlags(&ctx->small_copied, cudaEventDisableTiming));
    FH_CUDA(cudaStreamCreateWithFlags(&ctx->svd_side, cudaStreamNonBlocking));
    FH_CUDA(cudaEventCreateWithFlags(&ctx->svd_side_done, cudaEventDisableTiming));
  }
  // status words of this batch (checked by check_fact_status after the caller's next synchronisation)
  if (ctx->fact_status_pending) {
    FH_CUDA(cudaStreamSynchronize(ctx->stream));
    check_fact_status(ctx);
  }
  const int nstat = 2 * (int)order.size();
  if (nstat > ctx->fact_status_cap) {
    FH_CUDA(cudaStreamSynchronize(ctx->stream));
    if (ctx->d_fact_status) cudaFree(ctx->d_fact_status);
    if (ctx->h_fact_status) cudaFreeHost(ctx->h_fact_status);
    ctx->fact_status_cap = 2 * nstat + 256;
    FH_CUDA(cudaMalloc((void**)&ctx->d_fact_status, ctx->fact_status_cap * sizeof(int)));
    FH_CUDA(cudaMallocHost((void**)&ctx->h_fact_status, ctx->fact_status_cap * sizeof(int)));
  }
  int* const d_status = ctx->d_fact_status;
  if (nstat > 0) FH_CUDA(cudaMemsetAsync(d_status, 0, nstat * sizeof(int), ctx->stream));
  const int nord = (int)order.size();
  const int nw = (int)ctx->svd_workers.size();
  std::vector<int> idx;
  std::vector<SmallSvd> small;
  std::vector<MidSvd> mid;
  std::vector<SmallQr> small_qr;
  size_t small_smem = 0, small_qr_smem = 0;
  int64_t mid_v_total = 0;
  // fh_set_option(FH_OPT_SVD_MID_MAXN): 0 sends every matrix above the shared-memory route to cuSOLVER;
  // default 100 since the Gram route exists (measured: sweep 4.00 s with 100 / 104, 4.19 s with 128 / 160)
  const int mid_maxn = std::max(0, std::min(ctx->opt_svd_mid_maxn, MID_SVD_HARD_MAXN));
  const double mid_work = 1.5 * mid_maxn * (double)mid_maxn * mid_maxn;  // m n^2 bound: a long thin matrix would make its one CTA the critical path
  const int small_maxn = ctx->opt_svd_small_maxn;  // fh_set_option(FH_OPT_SVD_SMALL_MAXN)
  for (size_t i = 0; i < order.size(); ++i) {
    const int m = std::max(order[i]->nrow, order[i]->ncol), n = order[i]->k;
    if (!qr && n <= small_maxn && small_svd_bytes(m, n) <= SMALL_SVD_SMEM) {
      small.push_back(SmallSvd{order[i]->m_off, order[i]->u_off, order[i]->vt_off, order[i]->s_off, m, n, (int)i, 0});
      small_smem = std::max(small_smem, ((size_t)m * n + (size_t)n * n) * sizeof(cplx) + (size_t)n * sizeof(double));
    } else if (!qr && n <= mid_maxn && (double)m * n * n <= mid_work) {
      mid.push_back(MidSvd{order[i]->m_off, order[i]->u_off, order[i]->vt_off, order[i]->s_off, mid_v_total, m, n, (int)i, 0});
      mid_v_total += ((int64_t)n * n + 15) / 16 * 16;
    } else if (qr && order[i]->qn <= small_maxn && (size_t)order[i]->qm * order[i]->qn * sizeof(cplx) <= SMALL_QR_SMEM &&
               std::min(order[i]->qm, order[i]->qn) <= SMALL_QR_MAXK) {
      small_qr.push_back(SmallQr{order[i]->m_off, order[i]->r_dst, order[i]->qm, order[i]->qn, order[i]->r_ld,
                                 order[i]->r_transpose});
      small_qr_smem = std::max(small_qr_smem, (size_t)order[i]->qm * order[i]->qn * sizeof(cplx));
    } else {
      idx.push_back((int)i);
    }
  }
  // The worker streams fork from the main stream HERE, before the launch of the library's own small-matrix
  // kernel: that kernel (one CTA per matrix, a few tens of SMs) then runs on the main stream while the vendor
  // routines of the larger matrices run on the worker streams; the main stream joins them at the end.
  // one reservation for the descriptor tables of this call (reserve() rewinds the pool)
  ctx->pool_small.reserve(mid.size() * sizeof(MidSvd) + small.size() * sizeof(SmallSvd) +
                              small_qr.size() * sizeof(SmallQr) + 1024,
                          ctx->stream);
  MidSvd* d_mid = nullptr;
  int64_t mid_v_off = -1;
  if (!mid.empty()) {
    // heaviest first: the CTAs of the largest matrices start first
    std::stable_sort(mid.begin(), mid.end(), [](const MidSvd& a, const MidSvd& b) {
      return (double)a.m * a.n * a.n > (double)b.m * b.n * b.n;
    });
    const size_t need = mid.size() * sizeof(MidSvd);
    d_mid = (MidSvd*)ctx->pool_small.take(need);
    FH_CUDA(cudaMemcpyAsync(d_mid, stage_small_desc(ctx, mid.data(), need), need, cudaMemcpyHostToDevice, ctx->stream));
    FH_CUDA(cudaEventRecord(ctx->small_copied, ctx->stream));
    mid_v_off = ctx->alloc.alloc(mid_v_total);
  }
  if (!idx.empty() || !mid.empty()) {
    FH_CUDA(cudaEventRecord(ctx->svd_fork, ctx->stream));
    for (auto& w : ctx->svd_workers) FH_CUDA(cudaStreamWaitEvent(w.s, ctx->svd_fork, 0));
  }
  if (!mid.empty()) {
    FH_CUDA(cudaStreamWaitEvent(ctx->svd_side, ctx->svd_fork, 0));
    mid_svd_kernel<<<(int)mid.size(), 1024, 0, ctx->svd_side>>>(d_mid, buf, ctx->ptr(mid_v_off), dS, d_status);
    ++ctx->launches;
    ctx->svd_mid += (int64_t)mid.size();
    FH_CUDA(cudaGetLastError());
    FH_CUDA(cudaEventRecord(ctx->svd_side_done, ctx->svd_side));
  }
  // joins the side stream and returns the V scratch (stream-ordered: later users of that arena range are
  // enqueued on the main stream behind the wait)
  auto join_side = [&]() {
    if (mid.empty()) return;
    FH_CUDA(cudaStreamWaitEvent(ctx->stream, ctx->svd_side_done, 0));
    ctx->alloc.release(mid_v_off, mid_v_total);
  };
  if (!small_qr.empty()) {
    static bool qr_attr_done = false;
    if (!qr_attr_done) {
      FH_CUDA(cudaFuncSetAttribute(small_qr_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMALL_QR_SMEM));
      qr_attr_done = true;
    }
    const size_t need = small_qr.size() * sizeof(SmallQr);
    SmallQr* d_qr = (SmallQr*)ctx->pool_small.take(need);
    FH_CUDA(cudaMemcpyAsync(d_qr, stage_small_desc(ctx, small_qr.data(), need), need, cudaMemcpyHostToDevice, ctx->stream));
    FH_CUDA(cudaEventRecord(ctx->small_copied, ctx->stream));
    int qn_max = 0;  // one warp per trailing column of a Householder step
    for (const SmallQr& d : small_qr) qn_max = std::max(qn_max, d.n);
    const int qr_warps = qn_max <= 16 ? 8 : (qn_max <= 32 ? 16 : SMALL_QR_MAX_WARPS);
    small_qr_kernel<<<(int)small_qr.size(), 32 * qr_warps, small_qr_smem, ctx->stream>>>(d_qr, buf);
    ++ctx->launches;
    ctx->qr_small += (int64_t)small_qr.size();
    FH_CUDA(cudaGetLastError());
  }
  if (!small.empty()) {
    static bool attr_done = false;
    if (!attr_done) {
      FH_CUDA(cudaFuncSetAttribute(small_svd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   (int)SMALL_SVD_SMEM));
      attr_done = true;
    }
    const size_t need = small.size() * sizeof(SmallSvd);
    SmallSvd* d_small = (SmallSvd*)ctx->pool_small.take(need);
    FH_CUDA(cudaMemcpyAsync(d_small, stage_small_desc(ctx, small.data(), need), need, cudaMemcpyHostToDevice, ctx->stream));
    FH_CUDA(cudaEventRecord(ctx->small_copied, ctx->stream));
    // one warp per column pair of a tournament round: n / 2 pairs want up to 32 warps for the largest matrices
    int nmax = 0;
    for (const SmallSvd& d : small) nmax = std::max(nmax, d.n);
    const int warps = nmax <= 16 ? 8 : (nmax <= 32 ? 16 : SMALL_SVD_MAX_WARPS);
    small_svd_kernel<<<(int)small.size(), 32 * warps, small_smem, ctx->stream>>>(d_small, buf, dS, d_status);
    ++ctx->launches;
    ctx->svd_small += (int64_t)small.size();
    FH_CUDA(cudaGetLastError());
  }
  auto read_status = [&]() {
    if (nstat == 0) return;
    FH_CUDA(cudaMemcpyAsync(ctx->h_fact_status, d_status, nstat * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    ctx->fact_status_n = nstat;
    ctx->fact_status_pending = true;
  };
  if (idx.empty()) {
    join_side();
    read_status();
    return;
  }
  if (qr) ctx->qr_count += (int64_t)idx.size();
  auto cost = [&](int i) {
    const double m = std::max(order[i]->nrow, order[i]->ncol), n = order[i]->k;
    return m * n * n;
  };
  std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return cost(a) > cost(b); });
  // the mid-sized Gram-route sectors of the bond go through ONE batched eigensolver call on the last worker
  std::vector<int> gb;
  if (gram_minn > 0 && nw >= 2) {
    std::vector<int> rest;
    for (int i : idx) {
      const int n = order[i]->k;
      if (n >= gram_minn && n <= ctx->opt_svd_gram_batch_maxn) gb.push_back(i); else rest.push_back(i);
    }
    if (gb.size() >= 2) idx.swap(rest); else gb.clear();
  }
  const int nw_one = gb.empty() ? nw : nw - 1;  // workers that pull single matrices
  std::atomic<int> next{0};
  std::vector<std::string> errs(nw);
  std::vector<std::array<int64_t, 4>> counts(nw, std::array<int64_t, 4>{0, 0, 0, 0});
  auto body = [&](int wi) {
    try {
      FH_CUDA(cudaSetDevice(ctx->device));
      fh_ctx::SvdWorker& w = ctx->svd_workers[wi];
      for (;;) {
        const int i = next.fetch_add(1);
        if (i >= (int)idx.size()) break;
        if (qr) qr_one(w, *order[idx[i]], buf, d_status + idx[i], d_status + nord + idx[i]);
        else svd_one(w, *order[idx[i]], buf, dS, counts[wi].data(), d_status + idx[i], gram_minn);
      }
      FH_CUDA(cudaEventRecord(w.done, w.s));
    } catch (const std::exception& e) {
      errs[wi] = e.what();
      if (errs[wi].empty()) errs[wi] = "unknown error";
    }
  };
  const int nthreads = std::min<int>(nw_one, (int)idx.size());
  auto batch_body = [&]() {
    try {
      FH_CUDA(cudaSetDevice(ctx->device));
      fh_ctx::SvdWorker& w = ctx->svd_workers[nw - 1];
      gram_batch(w, order, gb, buf, dS, d_status);
      counts[nw - 1][3] += (int64_t)gb.size();
      FH_CUDA(cudaEventRecord(w.done, w.s));
    } catch (const std::exception& e) {
      errs[nw - 1] = e.what();
      if (errs[nw - 1].empty()) errs[nw - 1] = "unknown error";
    }
  };
  {
    std::vector<std::thread> th;
    if (!gb.empty()) th.emplace_back(batch_body);
    if (nthreads <= 1 && gb.empty()) {
      body(0);
    } else {
      for (int t = 0; t < std::max(1, nthreads); ++t) th.emplace_back(body, t);
    }
    for (auto& t : th) t.join();
  }
  // join every stream that was forked before reporting a worker's failure: nothing may still run on them
  std::string first_err;
  std::vector<int> used;
  for (int t = 0; t < std::max(1, nthreads); ++t) used.push_back(t);
  if (!gb.empty()) used.push_back(nw - 1);
  for (int t : used) {
    if (!errs[t].empty()) {
      if (first_err.empty()) first_err = errs[t];
      cudaStreamSynchronize(ctx->svd_workers[t].s);
      continue;
    }
    FH_CUDA(cudaStreamWaitEvent(ctx->stream, ctx->svd_workers[t].done, 0));
    for (int k = 0; k < 4; ++k) ctx->svd_count[k] += counts[t][k];
  }
  join_side();
  if (!first_err.empty()) throw FhError(FH_ECUDA, "sector SVD worker: " + first_err);
  read_status();
}

}  // namespace

void fh::check_fact_status(fh_ctx* ctx) {
  if (!ctx->fact_status_pending) return;
  ctx->fact_status_pending = false;
  for (int i = 0; i < ctx->fact_status_n; ++i) {
    const int v = ctx->h_fact_status[i];
    if (v == 0) continue;
    if (v == FACT_NOT_CONVERGED)
      throw FhError(FH_ECUDA, "sector SVD: one-sided Jacobi did not converge in " + std::to_string(JACOBI_MAX_SWEEPS) +
                                  " sweeps (matrix " + std::to_string(i) + " of the bond)");
    throw FhError(FH_ECUDA, "sector factorisation: cuSOLVER devInfo = " + std::to_string(v) + " (matrix " +
                                std::to_string(i % std::max(1, ctx->fact_status_n / 2)) + " of the bond)");
  }
}

// Reading A-6 (same rule as the oracle's, restated): sort all (s, sector, position) by s
// descending, ties by (sector index, position); drop s <= 1e-14 s_max; stop when the full
// dimension sum (2j+1) would exceed chi_max_full or the remaining tail weight is <= eps; keep >= 1.
static double truncate_rule(const std::vector<std::vector<double>>& sv, const std::vector<int>& mult, int chi_max,
                            double eps, std::vector<int>& keep) {
  struct It {
    double s;
    int c, p;
  };
  std::vector<It> items;
  for (size_t c = 0; c < sv.size(); ++c)
    for (size_t p = 0; p < sv[c].size(); ++p) items.push_back(It{sv[c][p], (int)c, (int)p});
  std::sort(items.begin(), items.end(), [](const It& a, const It& b) {
    if (a.s != b.s) return a.s > b.s;
    if (a.c != b.c) return a.c < b.c;
    return a.p < b.p;
  });
  double total = 0.0;
  for (const It& it : items) total += mult[it.c] * it.s * it.s;
  const double smax = items.empty() ? 0.0 : items[0].s;
  keep.assign(sv.size(), 0);
  int dim = 0, nk = 0;
  double kept = 0.0;
  for (const It& it : items) {
    if (nk >= 1) {
      if (it.s <= 1e-14 * smax) break;
      if (dim + mult[it.c] > chi_max) break;
      if (eps >= 0 && (total - kept) <= eps * total) break;
    }
    keep[it.c] += 1;
    dim += mult[it.c];
    kept += mult[it.c] * it.s * it.s;
    ++nk;
  }
  return total > 0 ? std::max(total - kept, 0.0) / total : 0.0;
}

// theta (layout th, device pointer) -> new A[i], A[i+1], bond[i+1].  direction +1: A[i] = U
// (left-canonical), A[i+1] = S V^H...; direction -1: A[i] = U S, A[i+1] = V^H... (right-canonical).
static void svd_split(fh_ctx* ctx, fh_mps* mps, int i, const BlockTensor& th, const cplx* theta, int direction,
                      const fh_params* prm) {
  const Bond& bl = mps->bond[i];
  const Bond& br = mps->bond[i + 2];
  // ---- group theta blocks by middle sector c
  std::map<Sector, SectorSvd> secs;
  for (size_t t = 0; t < th.keys.size(); ++t) {
    const Key& k = th.keys[t];
    const Sector c{k[3], k[4]};
    SectorSvd& S = secs[c];
    S.c = c;
    const Key rk{k[0], k[1], k[2], 0, 0, 0, 0, 0, 0, 0, 0, 0};
    const Key ck{k[5], k[6], k[7], 0, 0, 0, 0, 0, 0, 0, 0, 0};
    bool fr = false, fc = false;
    for (auto& r : S.rows) fr |= (r.first == rk);
    for (auto& cc : S.cols) fc |= (cc.first == ck);
    if (!fr) S.rows.push_back({rk, {0, th.rows[t]}});
    if (!fc) S.cols.push_back({ck, {0, th.cols[t]}});
  }
  int64_t cplx_total = 0, dbl_total = 0;
  std::vector<SectorSvd*> order;
  for (auto& e : secs) {
    SectorSvd& S = e.second;
    std::sort(S.rows.begin(), S.rows.end(), [](const auto& a, const auto& b) { return a.first < b.first; });
    std::sort(S.cols.begin(), S.cols.end(), [](const auto& a, const auto& b) { return a.first < b.first; });
    int n = 0;
    for (auto& r : S.rows) { r.second.first = n; n += r.second.second; }
    S.nrow = n;
    n = 0;
    for (auto& c : S.cols) { c.second.first = n; n += c.second.second; }
    S.ncol = n;
    S.k = std::min(S.nrow, S.ncol);
    S.transposed = S.nrow > S.ncol;  // cuSOLVER gesvd wants rows >= cols of the column-major matrix
    S.m_off = cplx_total;
    cplx_total += Arena::round_up((int64_t)S.nrow * S.ncol);
    S.u_off = cplx_total;
    cplx_total += Arena::round_up((int64_t)std::max(S.nrow, S.ncol) * S.k);
    S.vt_off = cplx_total;
    cplx_total += Arena::round_up((int64_t)S.k * std::min(S.nrow, S.ncol));
    S.s_off = dbl_total;
    dbl_total += (S.k + 1) / 2 * 2;
    order.push_back(&S);
  }
  const int64_t s_cplx = (dbl_total + 1) / 2;  // singular values live in the same scratch, as doubles
  const int64_t scratch_n = cplx_total + Arena::round_up(s_cplx);
  ArenaScratch scratch_mem(ctx, scratch_n);
  cplx* buf = scratch_mem.ptr();
  double* dS = reinterpret_cast<double*>(buf + cplx_total);
  cudaStream_t s = ctx->stream;

  // ---- pack (H8): M_c[(a,s1,al),(s2,b,be)] = theta[a,s1,c,s2,b] sqrt((2j_b+1)/(2j_c+1)); the vector already
  //      carries the sqrt(2j_b+1), so the copy only divides by sqrt(2j_c+1)
  ctx->timer_begin(T_PACK);
  launch_fill_zero(buf, cplx_total, s, &ctx->launches);
  std::vector<CopyBlk> blks;
  for (size_t t = 0; t < th.keys.size(); ++t) {
    const Key& k = th.keys[t];
    SectorSvd& S = secs[Sector{k[3], k[4]}];
    const Key rk{k[0], k[1], k[2], 0, 0, 0, 0, 0, 0, 0, 0, 0};
    const Key ck{k[5], k[6], k[7], 0, 0, 0, 0, 0, 0, 0, 0, 0};
    int ro = 0, co = 0;
    for (auto& r : S.rows) if (r.first == rk) ro = r.second.first;
    for (auto& c : S.cols) if (c.first == ck) co = c.second.first;
    CopyBlk b;
    b.src_off = th.off[t];
    b.rows = th.rows[t];
    b.cols = th.cols[t];
    b.ld_src = th.ld[t];
    b.scale = 1.0 / std::sqrt((double)(k[4] + 1));  // theta is held as sqrt(2 j_b + 1) theta
    b.pad = 0;
    if (!S.transposed) {  // row-major M_c (nrow x ncol)
      b.dst_off = S.m_off + (int64_t)ro * S.ncol + co;
      b.ld_dst = S.ncol;
      b.transpose_dst = 0;
    } else {  // row-major M_c^T (ncol x nrow)
      b.dst_off = S.m_off + (int64_t)co * S.nrow + ro;
      b.ld_dst = S.nrow;
      b.transpose_dst = 1;
    }
    blks.push_back(b);
  }
  ctx->pool_aux.reserve(blks.size() * sizeof(CopyBlk) + 4096, s);
  CopyBlk* d_blks = upload(ctx->pool_aux, blks, s);
  launch_copy_blocks(d_blks, (int)blks.size(), theta, buf, s, &ctx->launches);
  ctx->pack_bytes += 16 * cplx_total + 32 * th.nelem;  // zero fill of the work matrices + the scaled copy
  ctx->timer_end();

  // ---- block-wise SVD (H9): vendor routine, timed separately
  ctx->timer_begin(T_SVD);
  run_sector_svds(ctx, order, buf, dS);
  ctx->ensure_pinned((size_t)dbl_total + 2);
  FH_CUDA(cudaMemcpyAsync(ctx->h_pinned, dS, dbl_total * sizeof(double), cudaMemcpyDeviceToHost, s));
  FH_CUDA(cudaStreamSynchronize(s));
  ctx->timer_end();
  check_fact_status(ctx);

  // ---- truncation on the host (reading A-6)
  std::vector<std::vector<double>> sv;
  std::vector<int> mult, keep;
  for (SectorSvd* S : order) {
    sv.emplace_back(ctx->h_pinned + S->s_off, ctx->h_pinned + S->s_off + S->k);
    mult.push_back(S->c.tj + 1);
  }
  double disc = truncate_rule(sv, mult, prm->chi_max_full, prm->eps_trunc, keep);
  {
    // sectors factorised through the Gram matrix are accepted only if every KEPT singular value is large enough for
    // that route to be accurate (svd_one); the others are redone by the vendor SVD and the selection is repeated
    std::vector<SectorSvd*> redo;
    for (size_t x = 0; x < order.size(); ++x)
      if (order[x]->gram && keep[x] > 0 && sv[x][keep[x] - 1] < GRAM_SAFE_RATIO * sv[x][0]) redo.push_back(order[x]);
    if (!redo.empty()) {
      ctx->timer_begin(T_SVD);
      run_sector_svds(ctx, redo, buf, dS, false, false);
      FH_CUDA(cudaMemcpyAsync(ctx->h_pinned, dS, dbl_total * sizeof(double), cudaMemcpyDeviceToHost, s));
      FH_CUDA(cudaStreamSynchronize(s));
      ctx->timer_end();
      check_fact_status(ctx);
      ctx->svd_gram_redone += (int64_t)redo.size();
      for (size_t x = 0; x < order.size(); ++x)
        sv[x].assign(ctx->h_pinned + order[x]->s_off, ctx->h_pinned + order[x]->s_off + order[x]->k);
      disc = truncate_rule(sv, mult, prm->chi_max_full, prm->eps_trunc, keep);
    }
  }
  ctx->stat_disc = std::max(ctx->stat_disc, disc);
  Bond nb;
  for (size_t x = 0; x < order.size(); ++x) {
    order[x]->keep = keep[x];
    if (keep[x] > 0) {
      nb.sec.push_back(order[x]->c);
      nb.d.push_back(keep[x]);
    }
  }
  mps->bond[i + 1] = nb;
  mps->sval[i + 1].clear();
  for (size_t x = 0; x < order.size(); ++x)
    mps->sval[i + 1].insert(mps->sval[i + 1].end(), sv[x].begin(), sv[x].begin() + keep[x]);
  ctx->stat_chi = std::max(ctx->stat_chi, nb.chi_full());
  ctx->stat_su2 = std::max(ctx->stat_su2, nb.chi_su2());
  ctx->stat_dmax = std::max(ctx->stat_dmax, nb.dmax());

  // ---- unpack: A_i[a,s1,c] = U_c (x S), A_{i+1}[c,s2,b] = (S x) V_c^H sqrt((2j_c+1)/(2j_b+1))
  ctx->timer_begin(T_PACK);
  // With B = column-major (m x n) matrix given to gesvd, B = Ub S VTb:
  //   not transposed (B = M^T, m = ncol, n = nrow = k):  U_M[r][j] = VTb[j][r] -> memory r*k + j;
  //                                                     V^H[j][x]  = Ub[x][j]  -> memory j*m + x
  //   transposed     (B = M,   m = nrow, n = ncol = k):  U_M[r][j] = Ub[r][j]  -> memory j*m + r;
  //                                                     V^H[j][x]  = VTb[j][x] -> memory x*k + j
  for (SectorSvd* S : order) {
    if (S->keep == 0) continue;
    const int m = std::max(S->nrow, S->ncol), k = S->k;
    cplx* target;
    int nx;
    int64_t sj, sx;
    if (direction > 0) {  // scale V^H rows
      nx = S->ncol;
      if (!S->transposed) { target = buf + S->u_off; sj = m; sx = 1; } else { target = buf + S->vt_off; sj = 1; sx = k; }
    } else {  // scale U columns
      nx = S->nrow;
      if (!S->transposed) { target = buf + S->vt_off; sj = 1; sx = k; } else { target = buf + S->u_off; sj = m; sx = 1; }
    }
    const int64_t tot = (int64_t)S->keep * nx;
    scale_by_s_kernel<<<(int)std::min<int64_t>((tot + 255) / 256, 1184), 256, 0, s>>>(target, S->keep, nx, sj, sx,
                                                                                    dS + S->s_off);
    ++ctx->launches;
  }
  BlockTensor A1, A2;
  layout_site(bl, nb, A1);
  layout_site(nb, br, A2);
  ctx->free_tensor(mps->A[i]);
  ctx->free_tensor(mps->A[i + 1]);
  ctx->alloc_tensor(A1);
  ctx->alloc_tensor(A2);
  std::vector<CopyBlk> ub, vb;
  for (size_t t = 0; t < A1.keys.size(); ++t) {
    const Key& k = A1.keys[t];  // a(0,1) s1(2) c(3,4)
    SectorSvd& S = secs[Sector{k[3], k[4]}];
    const Key rk{k[0], k[1], k[2], 0, 0, 0, 0, 0, 0, 0, 0, 0};
    int ro = -1;
    for (auto& r : S.rows) if (r.first == rk) ro = r.second.first;
    FH_REQUIRE(ro >= 0, FH_ESTATE, "svd unpack: row block not found");
    const int m = std::max(S.nrow, S.ncol), kk = S.k;
    CopyBlk b;
    b.scale = 1.0;
    b.pad = 0;
    b.dst_off = A1.off[t];
    if (!S.transposed) {  // U_M row-major (nrow x k) in the VT buffer
      b.src_off = S.vt_off + (int64_t)ro * kk;
      b.rows = A1.rows[t];
      b.cols = S.keep;
      b.ld_src = kk;
      b.ld_dst = S.keep;
      b.transpose_dst = 0;
    } else {  // U buffer holds [j][r] with pitch m: copy rows j < keep, cols ro..ro+d_a, transposed
      b.src_off = S.u_off + ro;
      b.rows = S.keep;
      b.cols = A1.rows[t];
      b.ld_src = m;
      b.ld_dst = S.keep;
      b.transpose_dst = 1;
    }
    ub.push_back(b);
  }
  for (size_t t = 0; t < A2.keys.size(); ++t) {
    const Key& k = A2.keys[t];  // c(0,1) s2(2) b(3,4)
    SectorSvd& S = secs[Sector{k[0], k[1]}];
    const Key ck{k[2], k[3], k[4], 0, 0, 0, 0, 0, 0, 0, 0, 0};
    int co = -1;
    for (auto& c : S.cols) if (c.first == ck) co = c.second.first;
    FH_REQUIRE(co >= 0, FH_ESTATE, "svd unpack: column block not found");
    const int m = std::max(S.nrow, S.ncol), kk = S.k;
    CopyBlk b;
    b.scale = std::sqrt((double)(k[1] + 1) / (double)(k[4] + 1));
    b.pad = 0;
    b.dst_off = A2.off[t];
    if (!S.transposed) {  // V^H[j][x] at j*m + x in the U buffer
      b.src_off = S.u_off + co;
      b.rows = S.keep;
      b.cols = A2.cols[t];
      b.ld_src = m;
      b.ld_dst = A2.cols[t];
      b.transpose_dst = 0;
    } else {  // V^H[j][x] at x*k + j in the VT buffer: source rows x, cols j; write transposed
      b.src_off = S.vt_off + (int64_t)co * kk;
      b.rows = A2.cols[t];
      b.cols = S.keep;
      b.ld_src = kk;
      b.ld_dst = A2.cols[t];
      b.transpose_dst = 1;
    }
    vb.push_back(b);
  }
  ctx->pool_aux.reserve((ub.size() + vb.size()) * sizeof(CopyBlk) + 8192, s);
  CopyBlk* d_ub = upload(ctx->pool_aux, ub, s);
  CopyBlk* d_vb = upload(ctx->pool_aux, vb, s);
  launch_copy_blocks(d_ub, (int)ub.size(), buf, ctx->ptr(A1.base), s, &ctx->launches);
  launch_copy_blocks(d_vb, (int)vb.size(), buf, ctx->ptr(A2.base), s, &ctx->launches);
  ctx->pack_bytes += 32 * (A1.nelem + A2.nelem);
  FH_CUDA(cudaGetLastError());
  ctx->timer_end();
  mps->A[i] = A1;
  mps->A[i + 1] = A2;
}

// one local two-site update on bond (i, i+1)
static void local_update2(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, int i, double tau, int direction,
                          const fh_params* prm) {
  plan_heff(ctx, mpo, mps, i, 2);
  Plan& P = ctx->plan;
  const int64_t n = P.vec.nelem;
  const int m = prm->krylov_dim;
  const int64_t wn = (int64_t)(m + 2) * n;
  ArenaScratch work(ctx, wn);  // theta and the Krylov basis: returned also when a step below throws
  cplx* theta = work.ptr();
  cplx* V = theta + n;
  // merge (H8): theta[a,s1,c,s2,b] = A_i[a,s1,c] A_{i+1}[c,s2,b]; blocks whose c is not on the bond are zero
  {
    Stage st;
    emit_merge(mps->A[i], mps->A[i + 1], P.vec, st);
    ctx->pool_aux.reserve(stage_bytes(st) + 4096, ctx->stream);
    upload_stage(ctx->pool_aux, st, ctx->stream);
    ctx->timer_begin(T_PACK);
    launch_grouped_gemm(st, ctx->ptr(mps->A[i].base), ctx->ptr(mps->A[i + 1].base), theta, ctx->stream, &ctx->launches);
    ctx->timer_end();
  }
  expm_lanczos(ctx, theta, tau, m, prm->krylov_tol, V, prm->krylov_adapt_tol);
  BlockTensor th = P.vec;  // copy: svd_split re-plans nothing but keeps the layout alive
  svd_split(ctx, mps, i, th, theta, direction, prm);
}

static void local_update1(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, int i, double tau, const fh_params* prm) {
  plan_heff(ctx, mpo, mps, i, 1);
  Plan& P = ctx->plan;
  const int64_t n = P.vec.nelem;
  FH_REQUIRE(n == mps->A[i].nelem, FH_ESTATE, "one-site update: layout mismatch");
  const int m = prm->krylov_dim;
  const int64_t wn = (int64_t)(m + 1) * n;
  ArenaScratch work(ctx, wn);
  expm_lanczos(ctx, ctx->ptr(mps->A[i].base), tau, m, prm->krylov_tol, work.ptr(), prm->krylov_adapt_tol);
}

// ============================================================================ one-site TDVP (NEXT-1)
// Plan of the zero-site apply on the bond matrix C (layout Cl, keys {q, tj}) between Lenv and Renv.
// `bond` = index of the bond C lives on (cache key of the one-site sweeps' task lists, context.hpp).
static void plan_zero_site(fh_ctx* ctx, fh_mps* mps, int bond, const BlockTensor& Le, const BlockTensor& Re,
                           const BlockTensor& Cl) {
  Plan& P = ctx->plan;
  ctx->free_tensor(P.Z);
  if (P.ws_scratch >= 0) ctx->alloc.release(P.ws_scratch, P.ws_scratch_n);
  P.ws_scratch = -1;
  P.valid = false;
  P.io_ready = false;
  P.nsite = 0;
  P.site = -1;
  P.vec = Cl;
  P.vec.base = -1;
  std::vector<int> sig;
  const PlanCacheEntry* hit = nullptr;
  if (mps->cache.enabled) {
    sig_add(sig, Le);
    sig_add(sig, Re);
    sig_add(sig, Cl);
    hit = mps->cache.find(PC_HEFF0, bond, sig);
  }
  if (hit) {
    P.Z = hit->t1;
    P.st1 = hit->st1;
    P.st2 = hit->st2;
    P.chunks = hit->chunks;
  } else {
    emit_heff0(Le, Re, P.vec, P.Z, P.st1, P.st2);
    P.chunks.clear();
    const int cl = vec_chunk_len(P.vec.nelem);
    for (size_t i = 0; i < P.vec.keys.size(); ++i) {
      const int64_t n = (int64_t)P.vec.rows[i] * P.vec.cols[i];
      for (int64_t st = 0; st < n; st += cl)
        P.chunks.push_back(VecChunk{P.vec.off[i] + st, (int)std::min<int64_t>(cl, n - st), (float)(P.vec.keys[i][1] + 1)});
    }
    if (mps->cache.enabled) {
      if (PlanCacheEntry* e = mps->cache.store(PC_HEFF0, bond, std::move(sig))) {
        e->t1 = P.Z;
        e->st1 = P.st1;
        e->st2 = P.st2;
        e->chunks = P.chunks;
        mps->cache.account(e);
      }
    }
  }
  ctx->alloc_tensor(P.Z);
  P.ws_scratch_n = (int64_t)(P.st1.n_slots + P.st2.n_slots) * WS_SLOT_ELEMS;
  if (P.ws_scratch_n > 0) P.ws_scratch = ctx->alloc.alloc(P.ws_scratch_n);
  P.Lptr = ctx->ptr(Le.base);
  P.Rptr = ctx->ptr(Re.base);
  P.pair = WsPair();  // the zero-site apply always runs as warp units
  const size_t need = stage_bytes(P.st1) + stage_bytes(P.st2) + pair_bytes(P.pair) +
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

// Split the one-site tensor of site i without truncation (block-wise Householder QR per fused sector;
// measured 5-10x cheaper than the SVD drivers on these tall matrices):
//   direction +1: A_i[a,s,c] = Q[a,s,c] C[c],  Q left-canonical, C[c] = R (k_c x d_c, upper trapezoid) of the
//                 column-major stack M_c (rows (a,s,alpha)); bond i+1 gets dims k_c = min(rows, d_c)
//   direction -1: A_i[a,s,b] = C[a] Q[a,s,b],  Q right-canonical under the weights (2j_b+1)/(2j_a+1):
//                 QR of M~_a^T (M~_a = blocks side by side, scaled by sqrt of the weight): M~_a = R'^T Q'^T,
//                 C[a] = R'^T (d_a x k_a), Q = Q'^T with the weight undone; bond i gets dims k_a
// C is allocated in the arena (caller frees it).
static void split_site(fh_ctx* ctx, fh_mps* mps, int i, int direction, BlockTensor& C) {
  const BlockTensor Aold = mps->A[i];  // copy of the layout (device data stays where it is)
  const int gpos = direction > 0 ? 3 : 0;  // label position of the sector the blocks are grouped by
  std::map<Sector, SectorSvd> secs;
  struct Ref { int blk, ro, co; };
  std::map<Sector, std::vector<Ref>> refs;
  for (size_t t = 0; t < Aold.keys.size(); ++t) {
    const Key& k = Aold.keys[t];
    const Sector g{k[gpos], k[gpos + 1]};
    SectorSvd& S = secs[g];
    S.c = g;
    std::vector<Ref>& R = refs[g];
    if (R.empty()) S.nrow = S.ncol = 0;
    if (direction > 0) {  // stack rows (a, s): keys are sorted by (a, s) within a fixed c
      R.push_back(Ref{(int)t, S.nrow, 0});
      S.nrow += Aold.rows[t];
      S.ncol = Aold.cols[t];
    } else {  // side by side (s, b)
      R.push_back(Ref{(int)t, 0, S.ncol});
      S.ncol += Aold.cols[t];
      S.nrow = Aold.rows[t];
    }
  }
  int64_t cplx_total = 0;
  std::vector<SectorSvd*> order;
  Bond nb;
  for (auto& e : secs) {
    SectorSvd& S = e.second;
    S.k = std::min(S.nrow, S.ncol);
    S.keep = S.k;
    // the solver sees a column-major qm x qn matrix: M_c itself (+1) or M~_a^T (-1)
    S.qm = direction > 0 ? S.nrow : S.ncol;
    S.qn = direction > 0 ? S.ncol : S.nrow;
    S.m_off = cplx_total;
    cplx_total += Arena::round_up((int64_t)S.nrow * S.ncol);
    S.u_off = cplx_total;  // tau
    cplx_total += Arena::round_up(S.k);
    S.vt_off = S.s_off = 0;
    order.push_back(&S);
    nb.sec.push_back(S.c);
    nb.d.push_back(S.k);
  }
  const int64_t scratch = ctx->alloc.alloc(cplx_total);
  cplx* buf = ctx->ptr(scratch);
  cudaStream_t s = ctx->stream;
  // ---- new bond and layouts (dims are known before the factorisation: nothing is truncated)
  const int bpos = direction > 0 ? i + 1 : i;
  mps->bond[bpos] = nb;
  ctx->stat_chi = std::max(ctx->stat_chi, nb.chi_full());
  ctx->stat_su2 = std::max(ctx->stat_su2, nb.chi_su2());
  ctx->stat_dmax = std::max(ctx->stat_dmax, nb.dmax());
  BlockTensor Q;
  layout_site(mps->bond[i], mps->bond[i + 1], Q);
  C.clear();
  C.nlab = 2;
  for (SectorSvd* S : order) {
    if (direction > 0) C.add(Key{S->c.q, S->c.tj, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, S->k, S->ncol);
    else C.add(Key{S->c.q, S->c.tj, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, S->nrow, S->k);
  }
  C.finalize();
  ctx->alloc_tensor(Q);
  ctx->alloc_tensor(C);
  for (SectorSvd* S : order) {
    const int ci = C.find(Key{S->c.q, S->c.tj, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0});
    S->r_dst = ctx->ptr(C.base) + C.off[ci];
    S->r_ld = C.cols[ci];
    S->r_transpose = direction > 0 ? 0 : 1;  // -1: C[r][j] = R'[j][r]
  }
  // ---- pack: +1 column-major M_c (= row-major M_c^T), -1 row-major M~_a (= column-major M~_a^T)
  ctx->timer_begin(T_PACK);
  std::vector<CopyBlk> blks;
  for (auto& e : refs) {
    const SectorSvd& S = secs[e.first];
    for (const Ref& r : e.second) {
      const Key& k = Aold.keys[r.blk];
      CopyBlk b;
      b.src_off = Aold.off[r.blk];
      b.rows = Aold.rows[r.blk];
      b.cols = Aold.cols[r.blk];
      b.ld_src = Aold.cols[r.blk];
      b.pad = 0;
      if (direction > 0) {
        b.scale = 1.0;
        b.dst_off = S.m_off + (int64_t)r.co * S.nrow + r.ro;
        b.ld_dst = S.nrow;
        b.transpose_dst = 1;
      } else {
        b.scale = std::sqrt((double)(k[4] + 1) / (double)(k[1] + 1));
        b.dst_off = S.m_off + (int64_t)r.ro * S.ncol + r.co;
        b.ld_dst = S.ncol;
        b.transpose_dst = 0;
      }
      blks.push_back(b);
    }
  }
  ctx->pool_aux.reserve(blks.size() * sizeof(CopyBlk) + 4096, s);
  CopyBlk* d_blks = upload(ctx->pool_aux, blks, s);
  launch_copy_blocks(d_blks, (int)blks.size(), ctx->ptr(Aold.base), buf, s, &ctx->launches);
  ctx->timer_end();
  // ---- QR on the worker streams (R goes straight into C)
  ctx->timer_begin(T_SVD);
  run_sector_svds(ctx, order, buf, nullptr, true);
  ctx->timer_end();
  // ---- unpack Q (column-major qm x k at m_off)
  ctx->timer_begin(T_PACK);
  std::vector<CopyBlk> qb;
  for (auto& e : refs) {
    const SectorSvd& S = secs[e.first];
    const int k = S.k;
    for (const Ref& r : e.second) {
      const Key& key = Aold.keys[r.blk];
      const int qi = Q.find(key);
      FH_REQUIRE(qi >= 0, FH_ESTATE, "one-site split: block missing from the new layout");
      CopyBlk b;
      b.pad = 0;
      b.dst_off = Q.off[qi];
      b.ld_src = S.qm;
      b.rows = k;
      if (direction > 0) {  // Q[r][j] = Qcm[r + j m]: rows [ro, ro + d_a), read as (k x d_a) and transposed
        b.scale = 1.0;
        b.src_off = S.m_off + r.ro;
        b.cols = Aold.rows[r.blk];
        b.ld_dst = k;
        b.transpose_dst = 1;
      } else {  // Q[j][x] = Q'cm[x + j m]: columns [co, co + d_b) of the (k x m) row-major view
        b.scale = std::sqrt((double)(key[1] + 1) / (double)(key[4] + 1));
        b.src_off = S.m_off + r.co;
        b.cols = Aold.cols[r.blk];
        b.ld_dst = Aold.cols[r.blk];
        b.transpose_dst = 0;
      }
      qb.push_back(b);
    }
  }
  ctx->pool_aux.reserve(qb.size() * sizeof(CopyBlk) + 8192, s);
  CopyBlk* d_qb = upload(ctx->pool_aux, qb, s);
  launch_copy_blocks(d_qb, (int)qb.size(), buf, ctx->ptr(Q.base), s, &ctx->launches);
  FH_CUDA(cudaGetLastError());
  ctx->timer_end();
  ctx->free_tensor(mps->A[i]);
  mps->A[i] = Q;
  ctx->alloc.release(scratch, cplx_total);
}

// A_j <- C A_j (left) or A_j C (right) with the new bond dims already in mps->bond
static void absorb_bond(fh_ctx* ctx, fh_mps* mps, int j, const BlockTensor& C, bool left) {
  BlockTensor An;
  Stage st;
  const int kind = left ? PC_ABSORB_L : PC_ABSORB_R;
  std::vector<int> sig;
  const PlanCacheEntry* hit = nullptr;
  if (mps->cache.enabled) {
    sig_add(sig, C);
    sig_add(sig, mps->A[j]);
    sig_add(sig, mps->bond[j]);
    sig_add(sig, mps->bond[j + 1]);
    hit = mps->cache.find(kind, j, sig);
  }
  if (hit) {
    An = hit->t0;
    st = hit->st1;
  } else {
    layout_site(mps->bond[j], mps->bond[j + 1], An);
    emit_absorb(C, mps->A[j], An, left, st);
    if (mps->cache.enabled) {
      if (PlanCacheEntry* e = mps->cache.store(kind, j, std::move(sig))) {
        e->t0 = An;
        e->st1 = st;
        mps->cache.account(e);
      }
    }
  }
  ctx->alloc_tensor(An);
  ctx->pool_aux.reserve(stage_bytes(st) + 4096, ctx->stream);
  upload_stage(ctx->pool_aux, st, ctx->stream);
  ctx->timer_begin(T_PACK);
  if (left) launch_grouped_gemm(st, ctx->ptr(C.base), ctx->ptr(mps->A[j].base), ctx->ptr(An.base), ctx->stream, &ctx->launches);
  else launch_grouped_gemm(st, ctx->ptr(mps->A[j].base), ctx->ptr(C.base), ctx->ptr(An.base), ctx->stream, &ctx->launches);
  ctx->timer_end();
  FH_CUDA(cudaGetLastError());
  ctx->free_tensor(mps->A[j]);
  mps->A[j] = An;
}

static void zero_site_update(fh_ctx* ctx, fh_mps* mps, int bond, const BlockTensor& Le, const BlockTensor& Re,
                             BlockTensor& C, double tau, const fh_params* prm) {
  plan_zero_site(ctx, mps, bond, Le, Re, C);
  const int64_t n = C.nelem;
  const int m = prm->krylov_dim;
  const int64_t wn = (int64_t)(m + 1) * n;
  const int64_t woff = ctx->alloc.alloc(wn);
  expm_lanczos(ctx, ctx->ptr(C.base), tau, m, prm->krylov_tol, ctx->ptr(woff), prm->krylov_adapt_tol);
  ctx->alloc.release(woff, wn);
}

void fh::sweep1(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, double dt, const fh_params* prm) {
  const int L = mps->L;
  FH_REQUIRE(mpo->L == L, FH_EINVAL, "tdvp1_sweep: MPO and MPS lengths differ");
  for (int i = 0; i < L; ++i) FH_REQUIRE(mps->A[i].base >= 0, FH_ESTATE, "tdvp1_sweep: site tensor missing");
  for (int i = 1; i <= L; ++i) FH_REQUIRE(mps->Renv[i].base >= 0, FH_ESTATE, "tdvp1_sweep: right environments missing (centre must be at site 0)");
  ctx->stat_disc = 0.0;
  ctx->stat_chi = ctx->stat_su2 = ctx->stat_dmax = 0;
  const double tau = 0.5 * dt;
  // task lists are kept from one one-site sweep to the next (context.hpp, PlanCache); the guard switches the
  // cache off again on every exit so that no other entry point ever reads or fills it
  struct CacheScope {
    PlanCache& c;
    explicit CacheScope(PlanCache& cc) : c(cc) { c.enabled = c.max_bytes > 0; }
    ~CacheScope() { c.enabled = false; }
  } cache_scope(mps->cache);
  for (int i = 0; i < L; ++i) {  // left -> right
    local_update1(ctx, mpo, mps, i, tau, prm);
    if (i < L - 1) {
      BlockTensor C;
      split_site(ctx, mps, i, +1, C);
      do_env_update_left(ctx, mpo, mps, i);
      zero_site_update(ctx, mps, i + 1, mps->Lenv[i + 1], mps->Renv[i + 1], C, -tau, prm);
      absorb_bond(ctx, mps, i + 1, C, true);
      ctx->free_tensor(C);
    }
  }
  for (int i = L - 1; i >= 0; --i) {  // right -> left
    local_update1(ctx, mpo, mps, i, tau, prm);
    if (i > 0) {
      BlockTensor C;
      split_site(ctx, mps, i, -1, C);
      do_env_update_right(ctx, mpo, mps, i);
      zero_site_update(ctx, mps, i, mps->Lenv[i], mps->Renv[i], C, -tau, prm);
      absorb_bond(ctx, mps, i - 1, C, false);
      ctx->free_tensor(C);
    }
  }
  if (ctx->fact_status_pending) {
    FH_CUDA(cudaStreamSynchronize(ctx->stream));
    check_fact_status(ctx);
  }
}

void fh::sweep(fh_ctx* ctx, const fh_mpo* mpo, fh_mps* mps, double dt, const fh_params* prm) {
  const int L = mps->L;
  FH_REQUIRE(mpo->L == L, FH_EINVAL, "tdvp2_sweep: MPO and MPS lengths differ");
  for (int i = 0; i < L; ++i) FH_REQUIRE(mps->A[i].base >= 0, FH_ESTATE, "tdvp2_sweep: site tensor missing");
  for (int i = 2; i <= L; ++i) FH_REQUIRE(mps->Renv[i].base >= 0, FH_ESTATE, "tdvp2_sweep: right environments missing (centre must be at site 0)");
  mps->cache.clear();  // a two-site step changes the sector tables: the one-site task lists are stale
  ctx->stat_disc = 0.0;
  ctx->stat_chi = ctx->stat_su2 = ctx->stat_dmax = 0;
  const double tau = 0.5 * dt;
  // The task lists of the next two-site plan are emitted on a second host thread while this one runs the
  // backward one-site step: after the environment update every table and layout that plan reads is final.
  try {
    for (int i = 0; i < L - 1; ++i) {  // left -> right
      local_update2(ctx, mpo, mps, i, tau, +1, prm);
      do_env_update_left(ctx, mpo, mps, i);
      if (i < L - 2) {
        prefetch_plan2(ctx, mpo, mps, i + 1);
        local_update1(ctx, mpo, mps, i + 1, -tau, prm);
      }
    }
    for (int i = L - 2; i >= 0; --i) {  // right -> left
      local_update2(ctx, mpo, mps, i, tau, -1, prm);
      do_env_update_right(ctx, mpo, mps, i + 1);
      if (i > 0) {
        prefetch_plan2(ctx, mpo, mps, i - 1);
        local_update1(ctx, mpo, mps, i, -tau, prm);
      }
    }
  } catch (...) {
    prefetch_cancel(ctx);  // the job reads the state: it must be over before the caller may destroy it
    throw;
  }
  prefetch_cancel(ctx);
}

// H10: left norm environments N_{i+1}[c] = sum_{a,s} A^H N_i[a] A;  <O_i> = sum (2j_c+1) red(O)[s] Re Tr(A^H N A)
void fh::measure_local_impl(fh_ctx* ctx, const fh_mps* mps, double* n_i, double* sz_i, double* docc_i) {
  const int L = mps->L;
  cudaStream_t s = ctx->stream;
  BlockTensor N;
  N.nlab = 2;
  N.add(Key{0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, 1, 1);
  N.finalize();
  ctx->alloc_tensor(N);
  const cplx one = make_double2(1.0, 0.0);
  FH_CUDA(cudaMemcpyAsync(ctx->ptr(N.base), &one, sizeof(cplx), cudaMemcpyHostToDevice, s));
  for (int i = 0; i < L; ++i) {
    const BlockTensor& A = mps->A[i];
    FH_REQUIRE(A.base >= 0, FH_ESTATE, "measure_local: site tensor missing");
    BlockTensor Nn;
    Stage st1, st2;
    emit_norm_env(N, A, Nn, st1, st2);
    const int64_t xoff = ctx->alloc.alloc(A.nelem);
    ctx->alloc_tensor(Nn);
    std::vector<VecChunk> chunks;  // one or more chunks per block; weights applied on the host
    std::vector<int> chunk_blk;
    for (size_t b = 0; b < A.keys.size(); ++b) {
      const int64_t n = (int64_t)A.rows[b] * A.cols[b];
      for (int64_t o = 0; o < n; o += 8192) {
        chunks.push_back(VecChunk{A.off[b] + o, (int)std::min<int64_t>(8192, n - o), 1.0f});
        chunk_blk.push_back((int)b);
      }
    }
    ctx->pool_aux.reserve(stage_bytes(st1) + stage_bytes(st2) + chunks.size() * (sizeof(VecChunk) + 16) + 8192, s);
    upload_stage(ctx->pool_aux, st1, s);
    upload_stage(ctx->pool_aux, st2, s);
    VecChunk* d_chunks = upload(ctx->pool_aux, chunks, s);
    double* d_part = (double*)ctx->pool_aux.take(chunks.size() * 2 * sizeof(double));
    cplx* X = ctx->ptr(xoff);
    launch_grouped_gemm(st1, ctx->ptr(N.base), ctx->ptr(A.base), X, s, &ctx->launches);
    launch_wdot(d_chunks, (int)chunks.size(), ctx->ptr(A.base), X, d_part, nullptr, s, &ctx->launches);
    launch_grouped_gemm(st2, ctx->ptr(A.base), X, ctx->ptr(Nn.base), s, &ctx->launches);
    ctx->ensure_pinned(chunks.size() * 2 + 2);
    FH_CUDA(cudaMemcpyAsync(ctx->h_pinned, d_part, chunks.size() * 2 * sizeof(double), cudaMemcpyDeviceToHost, s));
    FH_CUDA(cudaStreamSynchronize(s));
    // expectation values of the diagonal one-site operators per site multiplet:
    //   SU2  (s = up, dn, pair): S^z = (1/2, -1/2, 0), n_up n_dn = (0, 0, 1/2) (half of the pair projector), n = (1, 1, 1)
    //        (the pair multiplet has <T^z> = 0 in a T_tot = 0 state, reading A-12);
    //   U1U1 (s = 0, up, dn, updn): S^z = (0, 1/2, -1/2, 0), n_up n_dn = (0, 0, 0, 1), n = (0, 1, 1, 2)
    static const double SZ[2][4] = {{0.5, -0.5, 0.0, 0.0}, {0.0, 0.5, -0.5, 0.0}};
    static const double DO[2][4] = {{0.0, 0.0, 0.5, 0.0}, {0.0, 0.0, 0.0, 1.0}};
    static const double NN[2][4] = {{1.0, 1.0, 1.0, 0.0}, {0.0, 1.0, 1.0, 2.0}};
    const int md = sym().id;
    double one_v = 0.0, sz = 0.0, pd = 0.0, nn = 0.0;
    for (size_t c = 0; c < chunks.size(); ++c) {
      const Key& k = A.keys[chunk_blk[c]];
      const double w = (k[4] + 1) * ctx->h_pinned[2 * c];
      one_v += w;
      sz += SZ[md][k[2]] * w;
      pd += DO[md][k[2]] * w;
      nn += NN[md][k[2]] * w;
    }
    // <n_i> = sum_s n_s w_s / <psi|psi>.  In the SU2 mode n_s = 1 for every multiplet (<n_i> = <1 + 2 T^z_i> and the
    // pair multiplet has <T^z_i> = 0 in a T_tot = 0 state, A-12): the numerator is the site's sum of multiplet
    // weights, the denominator the norm from the complete left-to-right contraction (filled in below), and the
    // ratio is 1 only if norm environments, multiplet weights and site tensors are consistent on every site.
    n_i[i] = nn;
    FH_REQUIRE(one_v > 0.0, FH_ESTATE, "measure_local: the state has zero weight on a site");
    sz_i[i] = sz / one_v;
    docc_i[i] = pd / one_v;
    ctx->alloc.release(xoff, A.nelem);
    ctx->free_tensor(N);
    N = Nn;
  }
  // <psi|psi> = the last norm environment (one 1 x 1 block of the total sector)
  double norm2 = 0.0;
  {
    ctx->ensure_pinned(2);
    FH_REQUIRE(N.nelem >= 1, FH_ESTATE, "measure_local: empty norm environment");
    FH_CUDA(cudaMemcpyAsync(ctx->h_pinned, ctx->ptr(N.base), sizeof(cplx), cudaMemcpyDeviceToHost, s));
    FH_CUDA(cudaStreamSynchronize(s));
    norm2 = ctx->h_pinned[0];
  }
  ctx->free_tensor(N);
  FH_REQUIRE(norm2 > 0.0, FH_ESTATE, "measure_local: the state has zero norm");
  for (int i = 0; i < L; ++i) n_i[i] /= norm2;
}
