// Microbenchmarks behind the roofline discussion of the fused tcgen05 kernels.  Built only into
// libhimuon_debug.so (-DHIMUON_DEBUG_STAGES); the product library gets an empty object.  Called by
// tests/test_gpu_microbench.py, whose printed table is kept as profiles/r2_microbench.txt.
//   mma_latency   cycles from the issue of n tcgen05.mma 128 x N x 16 (bf16, A in TMEM, fp32 accumulation, one dependent
//                 chain) to a polling thread seeing their tcgen05.commit: a fixed ~500 cycles + n x (N / 2) cycles.  A
//                 128 x 128 x 128 product therefore has a latency of ~1040 cycles for 512 cycles of tensor pipe.
//   tmem_read     tcgen05.ld.32x32b.x16 throughput of 8 warps reading a 128 x 128 fp32 accumulator (64 KB), alone and
//                 with a second accumulator being written by back-to-back MMAs: ~700 B per cycle and SM either way.
#ifdef HIMUON_DEBUG_STAGES
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "sm100_ptx.cuh"

namespace himuon {
namespace {
using namespace ptx;

template <int N>
__global__ void __launch_bounds__(128, 1) mma_latency_kernel(int n, int reps, long long* out) {
  extern __shared__ uint8_t smem_raw[];
  __shared__ uint32_t tb;
  __shared__ unsigned long long bar;
  const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const int warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) { mbar_init(smem_u32(&bar), 1); fence_mbar_init(); }
  if (warp == 0) tmem_alloc<512>(smem_u32(&tb));
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  if (warp == 1 && elect_one()) {
    const uint32_t idesc = make_idesc_bf16(128, N, 0, 0);
    uint32_t ph = 0;
    const long long t0 = clock64();
    for (int r = 0; r < reps; ++r) {
      for (int i = 0; i < n; ++i) {
        const int kk = i & 7;   // operand contents are irrelevant (whatever the shared memory holds)
        umma_bf16_ts(tb, tb + 128 + 8 * kk, make_smem_desc_sw128(smem0 + (kk >> 2) * 16384 + (kk & 3) * 32, 16, 1024), idesc, 1u);
      }
      umma_commit(smem_u32(&bar));
      mbar_wait(smem_u32(&bar), ph);
      ph ^= 1;
    }
    if (blockIdx.x == 0) out[0] = (clock64() - t0) / reps;
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tb);
}

// warps 0-7 read columns 256..383 (64 KB) `iters` times; warp 8 (with_mma) keeps 128 x 128 x 16 MMAs running into columns 0..127
__global__ void __launch_bounds__(320, 1) tmem_read_kernel(int iters, int with_mma, long long* out, float* sink) {
  extern __shared__ uint8_t smem_raw[];
  __shared__ uint32_t tb;
  __shared__ unsigned long long bar;
  __shared__ volatile int stop;
  const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const int warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) { mbar_init(smem_u32(&bar), 1); fence_mbar_init(); stop = 0; }
  if (warp == 0) tmem_alloc<512>(smem_u32(&tb));
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  float acc = 0.f;
  if (warp < 8) {
    const uint32_t base = tb + ((uint32_t)((warp & 3) * 32) << 16) + 256 + (warp >> 2) * 64;
    asm volatile("bar.sync 1, 256;");
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int c = 0; c < 64; c += 16) {
        uint32_t r[16];
        tmem_ld16(base + c, r);
        tmem_wait_ld();
        acc += __uint_as_float(r[0]) + __uint_as_float(r[15]);
      }
    }
    asm volatile("bar.sync 1, 256;");
    if (threadIdx.x == 0) {
      if (blockIdx.x == 0) out[0] = clock64() - t0;
      stop = 1;
    }
  } else if (warp == 8 && with_mma) {
    if (elect_one()) {
      const uint32_t idesc = make_idesc_bf16(128, 128, 0, 0);
      uint32_t ph = 0;
      long long n = 0;
      while (!stop) {
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)
          umma_bf16_ts(tb, tb + 128 + 8 * kk, make_smem_desc_sw128(smem0 + (kk >> 2) * 16384 + (kk & 3) * 32, 16, 1024), idesc, 1u);
        umma_commit(smem_u32(&bar));
        mbar_wait(smem_u32(&bar), ph);
        ph ^= 1;
        ++n;
      }
      if (blockIdx.x == 0) out[1] = n;
    }
    __syncwarp();
  }
  sink[blockIdx.x * blockDim.x + threadIdx.x] = acc;
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tb);
}

}  // namespace
}  // namespace himuon

// which = 0: mma_latency with N = 128, 1: with N = 64 (param = MMAs per commit) -> out[0] = cycles per commit;
// which = 2 / 3: tmem_read alone / with MMAs running (param = passes over 64 KB) -> out[0] = cycles, out[1] = products completed.
// out: 2 host long long.  Runs on every SM of the current device; returns a cudaError_t.
extern "C" int himuon_debug_microbench(int which, int param, long long* out) {
  using namespace himuon;
  long long* d = nullptr;
  float* sink = nullptr;
  int sms = 0, dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaError_t e = cudaMalloc(&d, 16);
  if (e != cudaSuccess) return (int)e;
  cudaMemset(d, 0, 16);
  const int smem = 100 * 1024;
  if (which == 0 || which == 1) {
    auto kern = which == 0 ? mma_latency_kernel<128> : mma_latency_kernel<64>;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    kern<<<sms, 128, smem>>>(param, 200, d);
  } else {
    cudaMalloc(&sink, (size_t)sms * 320 * 4);
    cudaFuncSetAttribute(tmem_read_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    tmem_read_kernel<<<sms, 320, smem>>>(param, which == 3 ? 1 : 0, d, sink);
  }
  e = cudaDeviceSynchronize();
  if (e == cudaSuccess) e = cudaMemcpy(out, d, 16, cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (sink) cudaFree(sink);
  return (int)e;
}
#endif  // HIMUON_DEBUG_STAGES
