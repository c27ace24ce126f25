// probe.cu -- fp64 peak probe behind wpcd_probe_fp64 (include/wpcd.h): the roofline denominator of the Jacobi stage is
// MEASURED in the bench run with this launch instead of being a constant.  Register-only chains:
// nothing but the fp64 datapath and the issue slots are exercised.
#include "wpcd_internal.cuh"

namespace {

constexpr int kProbeThreads = 512;
constexpr int kProbeCtasPerSm = 2;

__global__ void __launch_bounds__(kProbeThreads, kProbeCtasPerSm) k_probe_dfma(int iters, double* __restrict__ sink) {
  const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * (blockIdx.x + 1);
  double x0 = a, x1 = a + 1, x2 = a + 2, x3 = a + 3, x4 = a + 4, x5 = a + 5, x6 = a + 6, x7 = a + 7;
#pragma unroll 4
  for (int i = 0; i < iters; ++i) {
    x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
    x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
  }
  sink[(size_t)blockIdx.x * kProbeThreads + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

__global__ void __launch_bounds__(kProbeThreads, kProbeCtasPerSm) k_probe_dmma(int iters, double* __restrict__ sink) {
  const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * (blockIdx.x + 1);
  double d[8][2];
#pragma unroll
  for (int k = 0; k < 8; ++k) { d[k][0] = a + k; d[k][1] = b + k; }
#pragma unroll 2
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 8; ++k)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                   : "+d"(d[k][0]), "+d"(d[k][1])
                   : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += d[k][0] + d[k][1];
  sink[(size_t)blockIdx.x * kProbeThreads + threadIdx.x] = s;
}

}  // namespace

size_t wpcd_probe_sink(const WpcdHandle* h) { return (size_t)h->num_sms * kProbeCtasPerSm * kProbeThreads; }

int wpcd_probe_launch(WpcdHandle* h, int kind, int iters, double* d_sink, double* h_flops, cudaStream_t st) {
  const int grid = h->num_sms * kProbeCtasPerSm;
  const double threads = (double)grid * kProbeThreads;
  if (kind == 0) {
    k_probe_dfma<<<grid, kProbeThreads, 0, st>>>(iters, d_sink);
    *h_flops = threads * iters * 8.0 * 2.0;                       // 8 FMAs per thread and step
  } else {
    k_probe_dmma<<<grid, kProbeThreads, 0, st>>>(iters, d_sink);
    *h_flops = (threads / 32.0) * iters * 8.0 * (2.0 * 8 * 8 * 4);  // 8 m8n8k4 products per warp and step
  }
  return wpcd_check_cuda(h, cudaGetLastError(), "probe launch");
}
