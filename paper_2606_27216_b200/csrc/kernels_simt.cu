// fp32 path of the HiMuon hot path: one CTA owns one T x T tile, keeps X, A = X X^T and
// B = bA + cA^2 in shared memory for all K Newton-Schulz steps (Eq. 2.2-2.3; the
// "SRAM-resident" idea of PAPER.md:221) and does every product with fp32 FMAs.  The momentum update
// is fused into the tile load and the scaled, weight-decayed parameter write
// (Eq. 4.6) into the tile store, so W, G, M cross HBM once.
// Serves fp32 storage (config 1, tolerance 1e-4) and, on request (HIMUON_PATH_FP32), bf16 storage.
#include <cuda_bf16.h>

#include "himuon_internal.h"

namespace himuon {
namespace {

constexpr int kThreads = 256;

template <typename S> __device__ __forceinline__ float ld_elem(const S* p);
template <> __device__ __forceinline__ float ld_elem<float>(const float* p) { return *p; }
template <> __device__ __forceinline__ float ld_elem<__nv_bfloat16>(const __nv_bfloat16* p) { return __bfloat162float(*p); }
template <typename S> __device__ __forceinline__ void st_elem(S* p, float v);
template <> __device__ __forceinline__ void st_elem<float>(float* p, float v) { *p = v; }
template <> __device__ __forceinline__ void st_elem<__nv_bfloat16>(__nv_bfloat16* p, float v) { *p = __float2bfloat16_rn(v); }

// C(i,j) = sum_k P(i,k) * Q(j,k)   (NT)   or   sum_k P(i,k) * Q(k,j)   (NN); all T x T in smem, ld = T+1.
// Thread (ty,tx) of a 16x16 grid owns rows ty+16u, columns tx+16v.
template <int T, bool NN>
__device__ __forceinline__ void tile_gemm(const float* __restrict__ P, const float* __restrict__ Q,
                                          float (&acc)[(T / 16) * (T / 16)], int ty, int tx) {
  constexpr int TM = T / 16, LD = T + 1;
#pragma unroll
  for (int i = 0; i < TM * TM; ++i) acc[i] = 0.f;
#pragma unroll 4
  for (int k = 0; k < T; ++k) {
    float p[TM], q[TM];
#pragma unroll
    for (int u = 0; u < TM; ++u) p[u] = P[(ty + 16 * u) * LD + k];
#pragma unroll
    for (int v = 0; v < TM; ++v) q[v] = NN ? Q[k * LD + tx + 16 * v] : Q[(tx + 16 * v) * LD + k];
#pragma unroll
    for (int u = 0; u < TM; ++u)
#pragma unroll
      for (int v = 0; v < TM; ++v) acc[u * TM + v] = fmaf(p[u], q[v], acc[u * TM + v]);
  }
}

__device__ __forceinline__ float block_sum(float v, float* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  __syncthreads();
  if (l == 0) red[w] = v;
  __syncthreads();
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < kThreads / 32; ++i) s += red[i];
  return s;
}

template <int T, typename S>
__global__ void __launch_bounds__(kThreads, 1)
himuon_simt_kernel(const LayerDev* __restrict__ layers, const WorkItem* __restrict__ items, long long n_items,
                   int mode, himuon_hparams hp) {
  constexpr int TM = T / 16, LD = T + 1;
  extern __shared__ float smem[];
  float* X = smem;
  float* A = X + T * LD;
  float* B = A + T * LD;
  __shared__ float red[kThreads / 32];

  const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;

  for (long long it = blockIdx.x; it < n_items; it += gridDim.x) {
    WorkItem wi;
    if (items) wi = items[it];
    else { wi.layer = 0; wi.r = (int)it; wi.c = 0; wi.pad = 0; }
    const LayerDev L = layers[wi.layer];
    const int row0 = wi.r * T, col0 = wi.c * T;
    const S* G = reinterpret_cast<const S*>(L.g);
    S*       M = reinterpret_cast<S*>(L.m);
    S*       Wp = reinterpret_cast<S*>(L.w);

    // S1 momentum + S2 tile (zero padding) : PAPER.md:88-94, :51-53
    float ss = 0.f;
    for (int e = tid; e < T * T; e += kThreads) {
      const int i = e / T, j = e % T;
      const int gi = row0 + i, gj = col0 + j;
      float x = 0.f;
      if (gi < L.H && gj < L.W) {
        const float g = ld_elem<S>(G + (long long)gi * L.ld_g + gj);
        if (mode == MODE_STEP) {
          const float mp = ld_elem<S>(M + (long long)gi * L.ld_m + gj);
          const float mn = fmaf(hp.beta, mp, g);
          st_elem<S>(M + (long long)gi * L.ld_m + gj, mn);
          x = hp.nesterov ? fmaf(hp.beta, mn, g) : mn;
        } else {
          x = g;
        }
      }
      X[i * LD + j] = x;
      ss = fmaf(x, x, ss);
    }
    // S3 normalise: X0 = tile / (||tile||_F + eps); a zero tile stays zero
    const float tot = block_sum(ss, red);
    const float nrm = sqrtf(tot);
    const float inv = nrm > 0.f ? 1.f / (nrm + hp.eps) : 0.f;
    for (int e = tid; e < T * T; e += kThreads) X[(e / T) * LD + (e % T)] *= inv;
    __syncthreads();

    float* Xc = X;
    float* Ac = A;
    float  acc[TM * TM];
    // S4: K x (A = X X^T; B = bA + cA^2; X <- aX + BX)   Eq. (2.2)
    for (int k = 0; k < hp.K; ++k) {
      tile_gemm<T, false>(Xc, Xc, acc, ty, tx);
#pragma unroll
      for (int u = 0; u < TM; ++u)
#pragma unroll
        for (int v = 0; v < TM; ++v) Ac[(ty + 16 * u) * LD + tx + 16 * v] = acc[u * TM + v];
      __syncthreads();
      tile_gemm<T, false>(Ac, Ac, acc, ty, tx);   // A symmetric: A*A = A*A^T
#pragma unroll
      for (int u = 0; u < TM; ++u)
#pragma unroll
        for (int v = 0; v < TM; ++v) {
          const int idx = (ty + 16 * u) * LD + tx + 16 * v;
          B[idx] = fmaf(hp.c, acc[u * TM + v], hp.b * Ac[idx]);
        }
      __syncthreads();
      tile_gemm<T, true>(B, Xc, acc, ty, tx);
#pragma unroll
      for (int u = 0; u < TM; ++u)
#pragma unroll
        for (int v = 0; v < TM; ++v) {
          const int idx = (ty + 16 * u) * LD + tx + 16 * v;
          Ac[idx] = fmaf(hp.a, Xc[idx], acc[u * TM + v]);   // new X goes where A was
        }
      __syncthreads();
      float* t = Xc; Xc = Ac; Ac = t;
    }

    // S5 untile (crop) + S6 scaled, weight-decayed write: Eq. (4.6)
    const float tau = hp.scale_c * L.tau_base;
    const float keep = 1.f - hp.lr * hp.wd, step = hp.lr * tau;
    for (int e = tid; e < T * T; e += kThreads) {
      const int i = e / T, j = e % T;
      const int gi = row0 + i, gj = col0 + j;
      if (gi < L.H && gj < L.W) {
        const float u = Xc[i * LD + j];
        S* wp = Wp + (long long)gi * L.ld_w + gj;
        if (mode == MODE_STEP) st_elem<S>(wp, fmaf(keep, ld_elem<S>(wp), -step * u));
        else st_elem<S>(wp, u);
      }
    }
    __syncthreads();
  }
}

template <int T, typename S>
cudaError_t launch_t(const LaunchArgs& a, cudaStream_t s) {
  const size_t smem = 3ull * T * (T + 1) * sizeof(float);
  auto         kern = himuon_simt_kernel<T, S>;
  cudaError_t  e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int per_sm = 1;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kThreads, smem);
  if (e != cudaSuccess) return e;
  if (per_sm < 1) per_sm = 1;
  long long grid = (long long)device_sm_count() * per_sm;
  if (grid > a.n_items) grid = a.n_items;
  if (grid < 1) return cudaSuccess;
  kern<<<(unsigned)grid, kThreads, smem, s>>>(a.layers, a.items, a.n_items, a.mode, a.hp);
  return cudaGetLastError();
}

template <typename S>
cudaError_t launch_s(const LaunchArgs& a, cudaStream_t s) {
  switch (a.T) {
    case 16: return launch_t<16, S>(a, s);
    case 32: return launch_t<32, S>(a, s);
    case 64: return launch_t<64, S>(a, s);
    case 128: return launch_t<128, S>(a, s);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

// All layers of a launch share one storage dtype (buckets are keyed by dtype).
cudaError_t launch_simt(const LaunchArgs& a, cudaStream_t s) {
  return a.dtype == HIMUON_BF16 ? launch_s<__nv_bfloat16>(a, s) : launch_s<float>(a, s);
}

}  // namespace himuon
