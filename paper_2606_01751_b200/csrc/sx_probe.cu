// sx_probe.cu -- instruction-pipe rate probe (sx_probe_pipe in include/sparsex.h). Not part of the method: it
// measures, on the device it runs on, how many MUFU.EX2 / FFMA / FFMA2 lane-operations one SM retires per clock, the
// denominators of the scoring sweeps' roofline (stage (b) has one exponential per 256 flop: it is bound by the
// special-function pipe, not by the tensor pipe or HBM; S5). One CTA of 1024 threads per SM (8 warps per
// sub-partition), eight independent dependency chains per thread, cycles from clock64() around the loop.
#include "sx_internal.h"
#include "sx_ptx.cuh"

namespace sx {

template <int PIPE>
__global__ void __launch_bounds__(1024, 1)
probe_kernel(int iters, unsigned long long *__restrict__ cycles, float *__restrict__ sink) {
  float a[8];
  float2 a2[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    a[k] = 0.25f + 0.001f * (float)((threadIdx.x + 31 * k) & 255);
    a2[k] = make_float2(a[k], 0.5f * a[k]);
  }
  const float2 m2 = make_float2(0.999f, 1.001f), c2 = make_float2(1e-3f, -1e-3f);
  __syncthreads();
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      if (PIPE == 0) a[k] = ex2_approx(-a[k]);             // x -> 2^-x: stays in (0.5, 1)
      if (PIPE == 1) a[k] = fmaf(a[k], 0.999f, 1e-3f);      // scalar FFMA
      if (PIPE == 2) a2[k] = __ffma2_rn(a2[k], m2, c2);     // packed FFMA2: two fused multiply-adds per lane
      if (PIPE == 3) {                                      // the sweeps' mix: 3 MUFU.EX2 + 1 polynomial pair per 8 values
        if (k < 6) a[k] = ex2_approx(-a[k]);
        else if (k == 6) {
          const float2 e = ex2_poly2(make_float2(-a[6], -a[7]));
          a[6] = e.x;
          a[7] = e.y;
        }
      }
    }
  }
  const long long t1 = clock64();
  __syncthreads();
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += a[k] + a2[k].x + a2[k].y;
  if (s == 123456.789f) sink[0] = s;  // keeps the chains alive
  if (threadIdx.x == 0) cycles[blockIdx.x] = (unsigned long long)(t1 - t0);
}

sx_status launch_probe(int pipe, int iters, unsigned long long *cycles, int num_ctas, cudaStream_t st) {
  float *sink = reinterpret_cast<float *>(cycles + num_ctas);  // one spare word behind the cycle counts
  switch (pipe) {
    case 0: probe_kernel<0><<<num_ctas, 1024, 0, st>>>(iters, cycles, sink); break;
    case 1: probe_kernel<1><<<num_ctas, 1024, 0, st>>>(iters, cycles, sink); break;
    case 2: probe_kernel<2><<<num_ctas, 1024, 0, st>>>(iters, cycles, sink); break;
    case 3: probe_kernel<3><<<num_ctas, 1024, 0, st>>>(iters, cycles, sink); break;
    default: return set_error(SX_ERR_INVALID_ARG, "probe: pipe must be 0 (MUFU.EX2), 1 (FFMA), 2 (FFMA2) or 3 (sweep mix)");
  }
  return check_launch("probe_kernel");
}

}  // namespace sx
