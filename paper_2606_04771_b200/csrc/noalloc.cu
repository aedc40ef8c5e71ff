// fh_vec_wdot_static: the weighted inner product of two block vectors (F-6, the reduction of the Lanczos step, H6)
//     result = sum_b weight_b sum_{i in block b} conj(x_i) y_i
// for callers that may not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc.  fh_vec_wdot (api.cu) cuts the vector into chunks on the host, uploads the chunk table and takes its
// partial sums and its retirement counter from a pool of the context, which grows by cudaMalloc when it is too
// small.  This variant takes everything from the caller (vectors, block table and result are device pointers, the
// stream is the caller's) and keeps what it needs in between -- the prefix offsets of the blocks, one partial sum
// per CTA, the retirement counter -- in ONE file-scope array in device memory of fixed size:
//     NA_SCRATCH_BYTES = 8 (NA_MAX_BLOCKS + 1) + 16 NA_MAX_CTAS + 256  =  196 872 bytes,
// which every GPU that loads the library holds until the process exits.  It calls no cudaMalloc, no cudaFree and
// no allocating library routine, does not synchronise and copies nothing to the host: two kernel launches on the
// caller's stream.
//
// The array is shared by every call in the process and keeps the contents of the last call.  What has to start
// at zero (the retirement counter) is cleared by the first kernel of each call; prefix offsets and partial sums
// are written before they are read.  Two calls that overlap on one GPU (different streams without an ordering
// between them, or two host threads) race on the array: the caller serialises them.
//
// On the host the name of the array is a host-side stand-in, not a device address: its device address is taken
// once per device, with that device current, by cudaGetSymbolAddress (fh_static_setup, called by the entry
// point when the device has not been set up yet; call it yourself before starting a graph capture).
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>

#include "fh_b200.h"

namespace {

constexpr int NA_MAX_BLOCKS = FH_STATIC_MAX_BLOCKS;  // 16384 blocks
constexpr int NA_MAX_CTAS = 4096;
constexpr int NA_THREADS = 256;
constexpr size_t NA_OFF_PREFIX = 0;                                            // int64 [NA_MAX_BLOCKS + 1]
constexpr size_t NA_OFF_PARTIAL = sizeof(int64_t) * (NA_MAX_BLOCKS + 1);       // double [2 * NA_MAX_CTAS]
constexpr size_t NA_OFF_COUNTER = NA_OFF_PARTIAL + 16 * (size_t)NA_MAX_CTAS;   // unsigned, then the error word
constexpr size_t NA_SCRATCH_BYTES = NA_OFF_COUNTER + 256;
static_assert(NA_OFF_PARTIAL % 8 == 0 && NA_OFF_COUNTER % 8 == 0, "scratch regions must stay 8-byte aligned");
static_assert(NA_SCRATCH_BYTES == FH_STATIC_SCRATCH_BYTES, "the header states the size of the scratch array");

static __device__ __align__(256) unsigned char g_static_scratch[NA_SCRATCH_BYTES];

constexpr int NA_MAX_DEVICES = 64;
std::mutex g_mu;
unsigned char* g_scratch_ptr[NA_MAX_DEVICES] = {};  // device address of g_static_scratch, per device
thread_local char g_err[256] = "";

int fail(int code, const char* what, cudaError_t e = cudaSuccess) {
  if (e != cudaSuccess)
    snprintf(g_err, sizeof g_err, "%s: %s", what, cudaGetErrorString(e));
  else
    snprintf(g_err, sizeof g_err, "%s", what);
  return code;
}

__device__ __forceinline__ double warp_sum_na(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// One CTA: exclusive prefix sums of the block lengths (prefix[b] = first element of block b, prefix[nblk] = total),
// the retirement counter back to zero, and the status word: 1 if a length is negative or the lengths do not add
// up to n (the second kernel then writes NaN instead of a wrong number).
__global__ void __launch_bounds__(NA_THREADS) static_prefix_kernel(unsigned char* __restrict__ scratch, int nblk,
                                                                   const int64_t* __restrict__ blk_len, int64_t n) {
  int64_t* prefix = reinterpret_cast<int64_t*>(scratch + NA_OFF_PREFIX);
  unsigned* counter = reinterpret_cast<unsigned*>(scratch + NA_OFF_COUNTER);
  __shared__ int64_t tot[NA_THREADS];
  __shared__ int bad[NA_THREADS];
  const int per = (nblk + NA_THREADS - 1) / NA_THREADS;
  const int b0 = min(nblk, (int)threadIdx.x * per), b1 = min(nblk, b0 + per);
  int64_t s = 0;
  int neg = 0;
  for (int b = b0; b < b1; ++b) {
    neg |= blk_len[b] < 0;
    s += blk_len[b];
  }
  tot[threadIdx.x] = s;
  bad[threadIdx.x] = neg;
  __syncthreads();
  int64_t base = 0;
  for (int t = 0; t < (int)threadIdx.x; ++t) base += tot[t];
  for (int b = b0; b < b1; ++b) {
    prefix[b] = base;
    base += blk_len[b];
  }
  if (threadIdx.x == NA_THREADS - 1) {
    int any = 0;
    for (int t = 0; t < NA_THREADS; ++t) any |= bad[t];
    prefix[nblk] = base;
    counter[0] = 0u;
    counter[1] = (any || base != n) ? 1u : 0u;
  }
}

// CTA c sums its contiguous range [c * per_cta, (c + 1) * per_cta) of the vector; each thread walks the block
// table forward as its element index grows (binary search for the first block of the CTA's range).  The CTA that
// retires last adds the partial sums in index order with a fixed tree: the result does not depend on which CTA
// that is.
__global__ void __launch_bounds__(NA_THREADS) static_wdot_kernel(unsigned char* __restrict__ scratch, int nblk,
                                                                 const int32_t* __restrict__ blk_weight, int64_t n,
                                                                 int64_t per_cta, const double2* __restrict__ x,
                                                                 const double2* __restrict__ y,
                                                                 double* __restrict__ result) {
  const int64_t* prefix = reinterpret_cast<const int64_t*>(scratch + NA_OFF_PREFIX);
  double* partial = reinterpret_cast<double*>(scratch + NA_OFF_PARTIAL);
  unsigned* counter = reinterpret_cast<unsigned*>(scratch + NA_OFF_COUNTER);
  const int64_t e0 = (int64_t)blockIdx.x * per_cta;
  const int64_t e1 = min(n, e0 + per_cta);
  // last block whose first element is <= e0 (empty blocks in front of it are skipped by the walk below)
  int lo = 0, hi = nblk - 1;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (prefix[mid] <= e0) lo = mid; else hi = mid - 1;
  }
  int b = lo;
  int64_t bend = prefix[b + 1];
  double w = (double)blk_weight[b];
  double re = 0.0, im = 0.0;
  for (int64_t i = e0 + threadIdx.x; i < e1; i += NA_THREADS) {
    while (i >= bend && b < nblk - 1) {  // (the bound only matters for a block table the first kernel flagged)
      ++b;
      bend = prefix[b + 1];
      w = (double)blk_weight[b];
    }
    const double2 a = x[i], c = y[i];
    re += w * (a.x * c.x + a.y * c.y);
    im += w * (a.x * c.y - a.y * c.x);
  }
  __shared__ double sre[8], sim[8];
  __shared__ bool is_last;
  re = warp_sum_na(re);
  im = warp_sum_na(im);
  if ((threadIdx.x & 31) == 0) { sre[threadIdx.x >> 5] = re; sim[threadIdx.x >> 5] = im; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double r = 0.0, m = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { r += sre[i]; m += sim[i]; }
    partial[2 * blockIdx.x] = r;
    partial[2 * blockIdx.x + 1] = m;
    __threadfence();
    is_last = atomicAdd(counter, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  re = 0.0;
  im = 0.0;
  for (int i = threadIdx.x; i < (int)gridDim.x; i += NA_THREADS) {
    re += __ldcg(partial + 2 * i);
    im += __ldcg(partial + 2 * i + 1);
  }
  re = warp_sum_na(re);
  im = warp_sum_na(im);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) { sre[threadIdx.x >> 5] = re; sim[threadIdx.x >> 5] = im; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double r = 0.0, m = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { r += sre[i]; m += sim[i]; }
    if (counter[1]) r = m = __longlong_as_double(0x7ff8000000000000LL);  // bad block table: NaN, not a wrong number
    result[0] = r;
    result[1] = m;
  }
}

}  // namespace

extern "C" {

int fh_static_setup(void) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(FH_ECUDA, "fh_static_setup: cudaGetDevice", e);
  if (dev < 0 || dev >= NA_MAX_DEVICES) return fail(FH_EINVAL, "fh_static_setup: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_mu);
  if (g_scratch_ptr[dev]) return FH_OK;
  unsigned char* p = nullptr;
  e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
  if (e != cudaSuccess || !p) return fail(FH_ECUDA, "fh_static_setup: cudaGetSymbolAddress(g_static_scratch)", e);
  g_scratch_ptr[dev] = p;
  return FH_OK;
}

int fh_vec_wdot_static(int64_t n, int nblk, const int64_t* blk_len_dev, const int32_t* blk_weight_dev, const void* x_dev,
                       const void* y_dev, double* result_dev, void* stream) {
  if (n <= 0 || nblk <= 0 || !blk_len_dev || !blk_weight_dev || !x_dev || !y_dev || !result_dev)
    return fail(FH_EINVAL, "fh_vec_wdot_static: bad argument (n, nblk > 0 and six device pointers required)");
  if (nblk > NA_MAX_BLOCKS) {
    snprintf(g_err, sizeof g_err, "fh_vec_wdot_static: nblk = %d exceeds FH_STATIC_MAX_BLOCKS = %d (fixed scratch array)", nblk,
             NA_MAX_BLOCKS);
    return FH_EINVAL;
  }
  if (n > FH_STATIC_MAX_ELEMS) {
    snprintf(g_err, sizeof g_err, "fh_vec_wdot_static: n = %lld exceeds FH_STATIC_MAX_ELEMS = %lld", (long long)n,
             (long long)FH_STATIC_MAX_ELEMS);
    return FH_EINVAL;
  }
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(FH_ECUDA, "fh_vec_wdot_static: cudaGetDevice", e);
  if (dev < 0 || dev >= NA_MAX_DEVICES) return fail(FH_EINVAL, "fh_vec_wdot_static: device ordinal beyond 63");
  unsigned char* scratch;
  {
    std::lock_guard<std::mutex> lock(g_mu);
    scratch = g_scratch_ptr[dev];
  }
  if (!scratch) {
    const int rc = fh_static_setup();
    if (rc != FH_OK) return rc;
    std::lock_guard<std::mutex> lock(g_mu);
    scratch = g_scratch_ptr[dev];
  }
  // 1024 elements per CTA until NA_MAX_CTAS CTAs are in use, then longer ranges (a multiple of the CTA width)
  int64_t per_cta = 1024;
  if ((n + per_cta - 1) / per_cta > NA_MAX_CTAS) {
    per_cta = (n + NA_MAX_CTAS - 1) / NA_MAX_CTAS;
    per_cta = (per_cta + NA_THREADS - 1) / NA_THREADS * NA_THREADS;
  }
  const int ctas = (int)((n + per_cta - 1) / per_cta);
  cudaStream_t s = (cudaStream_t)stream;
  static_prefix_kernel<<<1, NA_THREADS, 0, s>>>(scratch, nblk, blk_len_dev, n);
  static_wdot_kernel<<<ctas, NA_THREADS, 0, s>>>(scratch, nblk, blk_weight_dev, n, per_cta, (const double2*)x_dev,
                                                 (const double2*)y_dev, result_dev);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(FH_ECUDA, "fh_vec_wdot_static: kernel launch", e);
  return FH_OK;
}

const char* fh_static_last_error(void) { return g_err; }

}  // extern "C"
