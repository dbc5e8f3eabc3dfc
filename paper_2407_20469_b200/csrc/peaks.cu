// peaks.cu - measured denominators of bench.py's roofline line ("to be measured by the harness with
// an FMA loop"): register-resident fp32 FFMA and FADD loops and a shared-memory read loop, timed with CUDA events
// on the given stream.  Test/bench-side entry (apic_measure_peak); not on the reconstruction path.
#include <cuda_runtime.h>

#include "../../include/apic.h"

namespace {

template <int MODE>
__global__ void __launch_bounds__(512) peak_alu_kernel(float* out, int iters, float seed) {
  constexpr int ILP = 8;
  float a[ILP];
#pragma unroll
  for (int i = 0; i < ILP; ++i) a[i] = seed + float(i) + float(threadIdx.x);
  const float b = seed * 0.5f, c = 1.0001f;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < ILP; ++i) {
      if (MODE == 0) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[i]) : "f"(c), "f"(b));
      else asm volatile("add.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(b));
    }
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < ILP; ++i) s += a[i];
  out[size_t(blockIdx.x) * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(512) peak_smem_kernel(float* out, int iters) {
  __shared__ float4 sh[2048];                                        // 32 KB
  for (int i = threadIdx.x; i < 2048; i += blockDim.x) sh[i] = make_float4(float(i), 1.f, 2.f, 3.f);
  __syncthreads();
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  int idx = threadIdx.x;
  const unsigned base = static_cast<unsigned>(__cvta_generic_to_shared(sh));
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      // eight DISTINCT entries per iteration (offsets k * 256 of a 2048-entry ring; k * 512 made k and k + 4 the same
      // address and let the compiler issue four loads for eight), each a volatile conflict-free LDS.128 that cannot be
      // merged or hoisted: the count of loads executed is the count the rate is computed from
      float4 v;
      asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                   : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                   : "r"(base + unsigned((idx + k * 256) & 2047) * 16u));
      acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
    }
    idx = (idx + 32) & 2047;
  }
  out[size_t(blockIdx.x) * blockDim.x + threadIdx.x] = acc.x + acc.y + acc.z + acc.w;
}

}  // namespace

extern "C" int apic_measure_peak(int what, double* per_second, void* cuda_stream) {
  if (!per_second || what < 0 || what > 2) return APIC_EINVAL;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return APIC_ECUDA;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int blocks = sms * 4, threads = 512, iters = 4096;
  float* out = nullptr;
  if (cudaMalloc(reinterpret_cast<void**>(&out), size_t(blocks) * threads * sizeof(float)) != cudaSuccess) return APIC_ENOMEM;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {                                 // first repetition warms up
    cudaEventRecord(e0, s);
    if (what == 0) peak_alu_kernel<0><<<blocks, threads, 0, s>>>(out, iters, 1.f);
    else if (what == 1) peak_alu_kernel<1><<<blocks, threads, 0, s>>>(out, iters, 1.f);
    else peak_smem_kernel<<<blocks, threads, 0, s>>>(out, iters);
    cudaEventRecord(e1, s);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(out); return APIC_ECUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  const double n = double(blocks) * threads * double(iters) * 8.0;
  if (what == 0) *per_second = 2.0 * n / (best * 1e-3);               // flop/s (an FMA = 2 flop)
  else if (what == 1) *per_second = n / (best * 1e-3);                // flop/s (adds)
  else *per_second = 16.0 * n / (best * 1e-3);                        // bytes/s read from shared memory
  return APIC_OK;
}
