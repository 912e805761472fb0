// Measured roofline denominators (measurement support, not on the hot path): nnp_measure_peaks runs four
// micro-benchmarks on the current device and returns what the hardware sustains for
//   [0] FP32 FFMA on the CUDA cores (TFLOP/s): 148 x 4 schedulers issuing independent FMA chains
//   [1] tcgen05.mma kind::tf32 from shared-memory operands (TFLOP/s): every SM issues M = 128, N = 256, K = 8
//       MMAs back to back into TMEM; no loads, no epilogue -- the rate the tensor pipe accepts TF32 work at
//   [2] reads of an L2-resident buffer (GB/s)
//   [3] reads of a buffer far larger than L2 (GB/s), for comparison with the driver's copy figure
// bench.py divides by these ("must be micro-benchmarked on the box before roofline fractions are
// quoted") instead of by derived numbers.
#include <cuda_runtime.h>
#include <stdint.h>

#include "nnp.h"

namespace {

__global__ void __launch_bounds__(512) ffma_kernel(float* out, int iters) {
  float a0 = threadIdx.x * 1e-3f, a1 = a0 + 1.f, a2 = a0 + 2.f, a3 = a0 + 3.f, a4 = a0 + 4.f, a5 = a0 + 5.f, a6 = a0 + 6.f,
        a7 = a0 + 7.f;
  const float b = 1.000001f, c = 1e-7f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      a0 = fmaf(a0, b, c); a1 = fmaf(a1, b, c); a2 = fmaf(a2, b, c); a3 = fmaf(a3, b, c);
      a4 = fmaf(a4, b, c); a5 = fmaf(a5, b, c); a6 = fmaf(a6, b, c); a7 = fmaf(a7, b, c);
    }
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

__global__ void __launch_bounds__(256) read_kernel(const float4* __restrict__ src, size_t n_vec, float* out, int reps) {
  float acc = 0.f;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (int r = 0; r < reps; ++r)
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i + 3 * stride < n_vec; i += 4 * stride) {
      const float4 v0 = __ldcg(src + i), v1 = __ldcg(src + i + stride), v2 = __ldcg(src + i + 2 * stride),
                   v3 = __ldcg(src + i + 3 * stride);
      acc += (v0.x + v1.y) + (v2.z + v3.w);
    }
  if (acc == 123.456f) out[0] = acc;  // keep the loads alive
}

__device__ __forceinline__ uint32_t s_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// One CTA per SM; warp 0 (converged, one elected lane) issues `n_mma` tf32 MMAs of 128 x 256 x 8 from two fixed
// shared-memory operand tiles into two alternating TMEM accumulators and waits for the last commit.
__global__ void __launch_bounds__(128, 1) mma_rate_kernel(int n_mma) {
  extern __shared__ __align__(1024) unsigned char smem_dyn[];
  unsigned char* base = smem_dyn + ((1024u - (s_u32(smem_dyn) & 1023u)) & 1023u);
  __shared__ __align__(8) uint64_t bar;
  __shared__ uint32_t tslot;
  for (int i = threadIdx.x; i < (16384 + 32768) / 4; i += blockDim.x) reinterpret_cast<float*>(base)[i] = 1.0f;
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(s_u32(&bar)) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  const int warp = threadIdx.x >> 5;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(s_u32(&tslot)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  if (warp == 0) {
    const uint32_t tmem = __shfl_sync(0xffffffffu, tslot, 0);
    uint32_t leader;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(leader));
    const uint32_t sa = __shfl_sync(0xffffffffu, s_u32(base), 0) >> 4;
    const uint64_t dk = (uint64_t)((16u >> 4) & 0x3FFF) << 16 | (uint64_t)((1024u >> 4) & 0x3FFF) << 32 | (1ull << 46) |
                        (2ull << 61);  // K-major, 128-byte swizzle
    const uint64_t da = dk | sa, db = dk | (sa + (16384u >> 4));
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((256u >> 3) << 17) | ((128u >> 4) << 24);
    if (leader) {
      for (int i = 0; i < n_mma; i += 4) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const uint32_t d = tmem + ((u & 1) ? 256u : 0u);
          const uint64_t a = da + 2 * u, b = db + 2 * u;
          asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                       ::"r"(d), "l"(a), "l"(b), "r"(idesc), "r"((uint32_t)(i > 1)) : "memory");
        }
      }
      asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(s_u32(&bar)) : "memory");
    }
    __syncwarp();
    uint32_t done;
    do {
      asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                   : "=r"(done) : "r"(s_u32(&bar)) : "memory");
    } while (!done);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tslot) : "memory");
}

template <typename F>
int time_ms(F launch, int reps, float* ms) {
  cudaEvent_t a, b;
  if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return -1;
  launch();  // warm-up
  float best = 1e30f;
  for (int r = 0; r < reps; ++r) {
    cudaEventRecord(a);
    launch();
    cudaEventRecord(b);
    if (cudaEventSynchronize(b) != cudaSuccess) return -1;
    float t = 0.f;
    cudaEventElapsedTime(&t, a, b);
    if (t < best) best = t;
  }
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  *ms = best;
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace

extern "C" int nnp_measure_peaks(double* peaks_host, int32_t n) {
  if (!peaks_host || n < 1) return NNP_ERR_INVALID_ARG;
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return NNP_ERR_CUDA;
  if (prop.major != 10) return NNP_ERR_UNSUPPORTED_ARCH;
  const int sms = prop.multiProcessorCount;
  double out[4] = {0, 0, 0, 0};
  float ms = 0.f;
  float* d_out = nullptr;
  if (cudaMalloc((void**)&d_out, sizeof(float) * (size_t)sms * 4 * 512) != cudaSuccess) return NNP_ERR_ALLOC;
  {  // FP32 FFMA: 4 CTAs of 512 threads per SM, 8 independent chains per thread
    const int iters = 4096;
    if (time_ms([&] { ffma_kernel<<<sms * 4, 512>>>(d_out, iters); }, 5, &ms)) { cudaFree(d_out); return NNP_ERR_CUDA; }
    out[0] = 2.0 * 64.0 * iters * (double)sms * 4 * 512 / (ms * 1e-3) / 1e12;
  }
  {  // tcgen05 kind::tf32
    const int n_mma = 8192;
    const int smem = 16384 + 32768 + 1024;
    if (cudaFuncSetAttribute((const void*)mma_rate_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess ||
        time_ms([&] { mma_rate_kernel<<<sms, 128, smem>>>(n_mma); }, 5, &ms)) { cudaFree(d_out); return NNP_ERR_CUDA; }
    out[1] = 2.0 * 128.0 * 256.0 * 8.0 * n_mma * (double)sms / (ms * 1e-3) / 1e12;
  }
  {  // L2-resident and DRAM reads
    const size_t small = (size_t)32 << 20, big = (size_t)2 << 30;
    float4* buf = nullptr;
    if (cudaMalloc((void**)&buf, big) != cudaSuccess) { cudaFree(d_out); return NNP_ERR_ALLOC; }
    cudaMemset(buf, 0, big);
    const int reps_small = 64;
    if (time_ms([&] { read_kernel<<<sms * 8, 256>>>(buf, small / 16, d_out, reps_small); }, 5, &ms) == 0)
      out[2] = (double)small * reps_small / (ms * 1e-3) / 1e9;
    if (time_ms([&] { read_kernel<<<sms * 8, 256>>>(buf, big / 16, d_out, 1); }, 5, &ms) == 0)
      out[3] = (double)big / (ms * 1e-3) / 1e9;
    cudaFree(buf);
  }
  cudaFree(d_out);
  for (int k = 0; k < n && k < 4; ++k) peaks_host[k] = out[k];
  return cudaDeviceSynchronize() == cudaSuccess ? NNP_OK : NNP_ERR_CUDA;
}
