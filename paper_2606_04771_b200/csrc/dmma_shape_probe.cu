// Not part of libfh_b200.so.  Compile-only probe behind DESIGN.md 6.1 / profiles/r2_zgemm_sass.md: what the FP64
// mma.sync shapes of PTX (m8n8k4, m16n8k4, m16n8k8, m16n8k16) lower to on sm_100a.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -cubin -o /tmp/dmma_shape_probe.cubin dmma_shape_probe.cu
//   cuobjdump -sass /tmp/dmma_shape_probe.cubin
extern "C" __global__ void probe_m8n8k4(double* out, const double* in) {
  double a = in[threadIdx.x], b = in[32 + threadIdx.x], c0 = 0.0, c1 = 0.0;
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
  out[2 * threadIdx.x] = c0;
  out[2 * threadIdx.x + 1] = c1;
}
extern "C" __global__ void probe_m16n8k4(double* out, const double* in) {
  double a0 = in[threadIdx.x], a1 = in[32 + threadIdx.x], b = in[64 + threadIdx.x], c[4] = {0, 0, 0, 0};
  asm volatile("mma.sync.aligned.m16n8k4.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};"
               : "+d"(c[0]), "+d"(c[1]), "+d"(c[2]), "+d"(c[3]) : "d"(a0), "d"(a1), "d"(b));
  for (int i = 0; i < 4; ++i) out[4 * threadIdx.x + i] = c[i];
}
extern "C" __global__ void probe_m16n8k8(double* out, const double* in) {
  double a[4], b[2], c[4] = {0, 0, 0, 0};
  for (int i = 0; i < 4; ++i) a[i] = in[32 * i + threadIdx.x];
  for (int i = 0; i < 2; ++i) b[i] = in[128 + 32 * i + threadIdx.x];
  asm volatile("mma.sync.aligned.m16n8k8.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+d"(c[0]), "+d"(c[1]), "+d"(c[2]), "+d"(c[3]) : "d"(a[0]), "d"(a[1]), "d"(a[2]), "d"(a[3]), "d"(b[0]), "d"(b[1]));
  for (int i = 0; i < 4; ++i) out[4 * threadIdx.x + i] = c[i];
}
extern "C" __global__ void probe_m16n8k16(double* out, const double* in) {
  double a[8], b[4], c[4] = {0, 0, 0, 0};
  for (int i = 0; i < 8; ++i) a[i] = in[32 * i + threadIdx.x];
  for (int i = 0; i < 4; ++i) b[i] = in[256 + 32 * i + threadIdx.x];
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7,%8,%9,%10,%11}, {%12,%13,%14,%15}, {%0,%1,%2,%3};"
      : "+d"(c[0]), "+d"(c[1]), "+d"(c[2]), "+d"(c[3])
      : "d"(a[0]), "d"(a[1]), "d"(a[2]), "d"(a[3]), "d"(a[4]), "d"(a[5]), "d"(a[6]), "d"(a[7]), "d"(b[0]), "d"(b[1]), "d"(b[2]), "d"(b[3]));
  for (int i = 0; i < 4; ++i) out[4 * threadIdx.x + i] = c[i];
}
