// Large tiles in TRUE fp32 arithmetic: fp32 storage, or HIMUON_PATH_FP32 on bf16 storage, at T >= 256 and on the
// full-matrix branch beyond the fp32 FMA kernel's tile sizes (the <= 1e-4 path of BASELINE.json; PAPER.md:424 uses an
// fp32 variant as its precision reference).  bf16 storage on the default path does NOT come here: its large tiles run
// on the hand-written tcgen05 GEMM path of kernels_lt.cu.  At these sizes every product of a Newton-Schulz step
// (Eq. 2.2) is a plain dense fp32 GEMM of library size, so the products go to cuBLAS (SGEMM,
// CUBLAS_COMPUTE_32F) and only the fused ends are kernels of this file:
//   k_prep   M' = beta M + G (stored), Ghat = G + beta M' | M' -> X (fp32 scratch),
//            per-block partial sums of squares (deterministic two-stage reduction)
//   k_scale  X <- X / (||Ghat||_F + eps), Phi_K(0) = 0
//   K x      A = X X^T (or X^T X for tall blocks);  B = b A + c A A;  B += a I;  X <- B X (or X B)
//   k_update W <- (1 - lr wd) W - lr tau X (Eq. 4.6; Phi mode: W <- X)
// A tile is addressed as a strided view of the parameter's own storage (no gather); the work items of a chunk
// are walked on the host, all launches asynchronous on the caller's stream; scratch (two fp32 copies of the tile, two
// r x r matrices, partial sums, 32 MB of cuBLAS workspace) lives in the caller's workspace.  cuBLAS is bound at run
// time (dlopen), so the library has no link-time dependency on it; if it cannot be found this path reports
// cudaErrorNotSupported.  One handle per device, enqueueing host threads serialised by a mutex.
#include <cublas_v2.h>
#include <cuda_bf16.h>
#include <dlfcn.h>

#include <algorithm>
#include <mutex>

#include "himuon_internal.h"

namespace himuon {
namespace {

// ---- cuBLAS, bound at run time -------------------------------------------------------------------------
struct Cublas {
  void* lib = nullptr;
  cublasStatus_t (*create)(cublasHandle_t*) = nullptr;
  cublasStatus_t (*set_stream)(cublasHandle_t, cudaStream_t) = nullptr;
  cublasStatus_t (*set_workspace)(cublasHandle_t, void*, size_t) = nullptr;
  cublasStatus_t (*gemm_ex)(cublasHandle_t, cublasOperation_t, cublasOperation_t, int, int, int, const void*,
                            const void*, cudaDataType, int, const void*, cudaDataType, int, const void*, void*,
                            cudaDataType, int, cublasComputeType_t, cublasGemmAlgo_t) = nullptr;
  cublasStatus_t (*gemm_batched)(cublasHandle_t, cublasOperation_t, cublasOperation_t, int, int, int, const void*,
                                 const void*, cudaDataType, int, long long, const void*, cudaDataType, int, long long,
                                 const void*, void*, cudaDataType, int, long long, int, cublasComputeType_t,
                                 cublasGemmAlgo_t) = nullptr;
  cublasHandle_t handles[64] = {};   // one per device ordinal, created on first use on that device
  cublasHandle_t handle = nullptr;   // the current device's, set by acquire() under `mu`
  std::mutex mu;                     // a handle carries a stream and a workspace: one enqueueing host thread at a time
  bool ok = false;
  // Call with `mu` held: select (create if needed) the handle of the current device.
  bool acquire() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return false;
    if (!handles[dev] && create(&handles[dev]) != CUBLAS_STATUS_SUCCESS) { handles[dev] = nullptr; return false; }
    handle = handles[dev];
    return true;
  }
};

Cublas& cublas() {
  static Cublas c;
  static std::once_flag once;
  std::call_once(once, [] {
    for (const char* name : {"libcublas.so.12", "libcublas.so", "/usr/local/cuda/lib64/libcublas.so.12"}) {
      c.lib = dlopen(name, RTLD_NOW | RTLD_GLOBAL);
      if (c.lib) break;
    }
    if (!c.lib) return;
    c.create = reinterpret_cast<decltype(c.create)>(dlsym(c.lib, "cublasCreate_v2"));
    c.set_stream = reinterpret_cast<decltype(c.set_stream)>(dlsym(c.lib, "cublasSetStream_v2"));
    c.set_workspace = reinterpret_cast<decltype(c.set_workspace)>(dlsym(c.lib, "cublasSetWorkspace_v2"));
    c.gemm_ex = reinterpret_cast<decltype(c.gemm_ex)>(dlsym(c.lib, "cublasGemmEx"));
    c.gemm_batched = reinterpret_cast<decltype(c.gemm_batched)>(dlsym(c.lib, "cublasGemmStridedBatchedEx"));
    c.ok = c.create && c.set_stream && c.set_workspace && c.gemm_ex && c.gemm_batched;
  });
  return c;
}

// ---- elementwise ends -------------------------------------------------------------------------------------
constexpr int kEwThreads = 256;
constexpr int kEwBlocks = 1024;          // fixed grid: the partial sums of squares have a fixed summation order

template <typename S> __device__ __forceinline__ float ld_elem(const S* p);
template <> __device__ __forceinline__ float ld_elem<float>(const float* p) { return *p; }
template <> __device__ __forceinline__ float ld_elem<__nv_bfloat16>(const __nv_bfloat16* p) { return __bfloat162float(*p); }
template <typename S> __device__ __forceinline__ void st_elem(S* p, float v);
template <> __device__ __forceinline__ void st_elem<float>(float* p, float v) { *p = v; }
template <> __device__ __forceinline__ void st_elem<__nv_bfloat16>(__nv_bfloat16* p, float v) { *p = __float2bfloat16_rn(v); }

// One h x w block of a row-major matrix with leading dimension ld.
template <typename S>
struct View {
  S* p;
  long long ld;
};

template <typename S>
__global__ void __launch_bounds__(kEwThreads)
k_prep(View<const S> G, View<S> M, float* __restrict__ X, float* __restrict__ partial, int h, int w, int step_mode,
       float beta, int nesterov) {
  const long long n = (long long)h * w;
  float ss = 0.f;
  for (long long i = (long long)blockIdx.x * kEwThreads + threadIdx.x; i < n; i += (long long)gridDim.x * kEwThreads) {
    const int r = (int)(i / w), c = (int)(i - (long long)r * w);
    const float g = ld_elem(G.p + r * G.ld + c);
    float x = g;
    if (step_mode) {
      const float m = fmaf(beta, ld_elem(M.p + r * M.ld + c), g);
      st_elem(M.p + r * M.ld + c, m);
      x = nesterov ? fmaf(beta, m, g) : m;
    }
    X[i] = x;
    ss = fmaf(x, x, ss);
  }
  __shared__ float red[kEwThreads / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
  __syncthreads();
  if (threadIdx.x == 0) {
    float t = 0.f;
#pragma unroll
    for (int i = 0; i < kEwThreads / 32; ++i) t += red[i];
    partial[blockIdx.x] = t;
  }
}

// Every block sums the same partials in the same order, then scales its share of X.
__global__ void __launch_bounds__(kEwThreads)
k_scale(float* __restrict__ X, const float* __restrict__ partial, int n_partial, long long n, float eps) {
  __shared__ float red[kEwThreads / 32];
  __shared__ float inv_s;
  float t = 0.f;
  for (int i = threadIdx.x; i < n_partial; i += kEwThreads) t += partial[i];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = t;
  __syncthreads();
  if (threadIdx.x == 0) {
    float tot = 0.f;
#pragma unroll
    for (int i = 0; i < kEwThreads / 32; ++i) tot += red[i];
    const float nrm = sqrtf(tot);
    inv_s = nrm > 0.f ? 1.f / (nrm + eps) : 0.f;
  }
  __syncthreads();
  const float inv = inv_s;
  for (long long i = (long long)blockIdx.x * kEwThreads + threadIdx.x; i < n; i += (long long)gridDim.x * kEwThreads) X[i] *= inv;
}

__global__ void k_add_diag(float* __restrict__ B, int r, float a) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < r) B[(long long)i * r + i] += a;
}

template <typename S>
__global__ void __launch_bounds__(kEwThreads)
k_update(View<S> W, const float* __restrict__ X, int h, int w, int step_mode, float keep, float stepsz) {
  const long long n = (long long)h * w;
  for (long long i = (long long)blockIdx.x * kEwThreads + threadIdx.x; i < n; i += (long long)gridDim.x * kEwThreads) {
    const int r = (int)(i / w), c = (int)(i - (long long)r * w);
    S* p = W.p + r * W.ld + c;
    const float x = X[i];
    st_elem(p, step_mode ? fmaf(keep, ld_elem(p), stepsz * x) : x);
  }
}

// ---- batched form for uniform tiles (T = 256 / 512): grid (kTileBlocks, tiles of the sub-batch) ----------------
// The tiles of a sub-batch are staged as dense, zero-padded T x T fp32 matrices (the
// paper's batched buffers, here bounded by a scratch budget and refilled sub-batch by sub-batch).
constexpr int kTileBlocks = 32;

template <typename S>
__global__ void __launch_bounds__(kEwThreads)
k_prep_b(const LayerDev* __restrict__ layers, const WorkItem* __restrict__ items, float* __restrict__ X,
         float* __restrict__ partial, int Th, int Tw, long long stride, int step_mode, float beta, int nesterov) {
  const WorkItem wi = items[blockIdx.y];
  const LayerDev L = layers[wi.layer];
  const int row0 = wi.r * Th, col0 = wi.c * Tw;
  const S* G = reinterpret_cast<const S*>(L.g);
  S* M = reinterpret_cast<S*>(L.m);
  float* Xt = X + (long long)blockIdx.y * stride;
  float ss = 0.f;
  for (int i = blockIdx.x * kEwThreads + threadIdx.x; i < Th * Tw; i += kTileBlocks * kEwThreads) {
    const int r = i / Tw, c = i - r * Tw;
    float x = 0.f;
    if (row0 + r < L.H && col0 + c < L.W) {
      const float g = ld_elem(G + (long long)(row0 + r) * L.ld_g + col0 + c);
      x = g;
      if (step_mode) {
        S* pm = M + (long long)(row0 + r) * L.ld_m + col0 + c;
        const float m = fmaf(beta, ld_elem(pm), g);
        st_elem(pm, m);
        x = nesterov ? fmaf(beta, m, g) : m;
      }
    }
    Xt[i] = x;
    ss = fmaf(x, x, ss);
  }
  __shared__ float red[kEwThreads / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
  __syncthreads();
  if (threadIdx.x == 0) {
    float t = 0.f;
#pragma unroll
    for (int i = 0; i < kEwThreads / 32; ++i) t += red[i];
    partial[blockIdx.y * kTileBlocks + blockIdx.x] = t;
  }
}

__global__ void __launch_bounds__(kEwThreads)
k_scale_b(float* __restrict__ X, const float* __restrict__ partial, int n, long long stride, float eps) {
  float tot = 0.f;
#pragma unroll
  for (int i = 0; i < kTileBlocks; ++i) tot += partial[blockIdx.y * kTileBlocks + i];   // same order in every thread
  const float nrm = sqrtf(tot);
  const float inv = nrm > 0.f ? 1.f / (nrm + eps) : 0.f;
  float* Xt = X + (long long)blockIdx.y * stride;
  for (int i = blockIdx.x * kEwThreads + threadIdx.x; i < n; i += kTileBlocks * kEwThreads) Xt[i] *= inv;
}

__global__ void k_add_diag_b(float* __restrict__ B, int T, long long stride, float a) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < T) B[(long long)blockIdx.y * stride + (long long)i * T + i] += a;
}

template <typename S>
__global__ void __launch_bounds__(kEwThreads)
k_update_b(const LayerDev* __restrict__ layers, const WorkItem* __restrict__ items, const float* __restrict__ X, int Th,
           int Tw, long long stride, int step_mode, float keep, float lr_scale) {
  const WorkItem wi = items[blockIdx.y];
  const LayerDev L = layers[wi.layer];
  const int row0 = wi.r * Th, col0 = wi.c * Tw;
  S* W = reinterpret_cast<S*>(L.w);
  const float* Xt = X + (long long)blockIdx.y * stride;
  const float stepsz = lr_scale * L.tau_base;
  for (int i = blockIdx.x * kEwThreads + threadIdx.x; i < Th * Tw; i += kTileBlocks * kEwThreads) {
    const int r = i / Tw, c = i - r * Tw;
    if (row0 + r < L.H && col0 + c < L.W) {
      S* p = W + (long long)(row0 + r) * L.ld_w + col0 + c;
      st_elem(p, step_mode ? fmaf(keep, ld_elem(p), stepsz * Xt[i]) : Xt[i]);
    }
  }
}

constexpr size_t kCublasWs = 32u << 20;
size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace

// Scratch bytes for one h x w block: X, X2 (fp32), A, B (r x r fp32, r = min(h, w)), partial sums, cuBLAS workspace.
size_t gemm_path_scratch_bytes(int h, int w) {
  const size_t r = (size_t)std::min(h, w);
  return 2 * align256((size_t)h * w * 4) + 2 * align256(r * r * 4) + align256(kEwBlocks * 4) + kCublasWs;
}

// Scratch bytes per tile of the batched form: X, X2, A, B (T x T fp32 each) and the partial sums.
size_t gemm_path_fixed_bytes() { return kCublasWs; }
size_t gemm_path_batch_item_bytes(int Th, int Tw) {
  const size_t r = (size_t)std::min(Th, Tw);
  return 2 * align256((size_t)Th * Tw * 4) + 2 * align256(r * r * 4) + align256(kTileBlocks * 4);
}

namespace {

// One sub-batch of nb uniform Th x Tw tiles, staged zero-padded (items_dev / layers_dev: device copies of the work
// items and of the layer table).  Gram matrix on the short side of the tile.
template <typename S>
cudaError_t run_batch(const LayerDev* layers_dev, const WorkItem* items_dev, int nb, int Th, int Tw, int mode,
                      const himuon_hparams& hp, char* scratch, cudaStream_t s, long long* launches) {
  Cublas& cb = cublas();
  const int r = std::min(Th, Tw);
  const size_t xb = align256((size_t)Th * Tw * 4), ab = align256((size_t)r * r * 4);
  float* X = reinterpret_cast<float*>(scratch);
  float* X2 = reinterpret_cast<float*>(scratch + (size_t)nb * xb);
  float* A = reinterpret_cast<float*>(scratch + 2 * (size_t)nb * xb);
  float* B = reinterpret_cast<float*>(scratch + 2 * (size_t)nb * xb + (size_t)nb * ab);
  float* partial = reinterpret_cast<float*>(scratch + 2 * (size_t)nb * (xb + ab));
  void* cws = scratch + 2 * (size_t)nb * (xb + ab) + (size_t)nb * align256(kTileBlocks * 4);
  const bool step_mode = (mode == MODE_STEP);
  const long long sx = (long long)(xb / 4), sa = (long long)(ab / 4);
  const int h = Th, w = Tw;
  const dim3 grid(kTileBlocks, nb);
  k_prep_b<S><<<grid, kEwThreads, 0, s>>>(layers_dev, items_dev, X, partial, Th, Tw, sx, step_mode ? 1 : 0, hp.beta, hp.nesterov);
  k_scale_b<<<grid, kEwThreads, 0, s>>>(X, partial, Th * Tw, sx, hp.eps);
  *launches += 2;
  if (hp.K > 0) {
    if (cb.set_stream(cb.handle, s) != CUBLAS_STATUS_SUCCESS) return cudaErrorUnknown;
    if (cb.set_workspace(cb.handle, cws, kCublasWs) != CUBLAS_STATUS_SUCCESS) return cudaErrorUnknown;
  }
  const cublasComputeType_t ct = CUBLAS_COMPUTE_32F;   // this path is the true-fp32 one for either storage type
  const float one = 1.f, zero = 0.f;
  // Row-major X (h x w, ld = w) is the column-major w x h matrix Xc = X^T with leading dimension w (see run_one).
  for (int k = 0; k < hp.K; ++k) {
    cublasStatus_t st;
    if (h <= w)
      st = cb.gemm_batched(cb.handle, CUBLAS_OP_T, CUBLAS_OP_N, h, h, w, &one, X, CUDA_R_32F, w, sx, X, CUDA_R_32F, w, sx,
                           &zero, A, CUDA_R_32F, r, sa, nb, ct, CUBLAS_GEMM_DEFAULT);
    else
      st = cb.gemm_batched(cb.handle, CUBLAS_OP_N, CUBLAS_OP_T, w, w, h, &one, X, CUDA_R_32F, w, sx, X, CUDA_R_32F, w, sx,
                           &zero, A, CUDA_R_32F, r, sa, nb, ct, CUBLAS_GEMM_DEFAULT);
    if (st != CUBLAS_STATUS_SUCCESS) return cudaErrorUnknown;
    cudaError_t e = cudaMemcpyAsync(B, A, (size_t)nb * ab, cudaMemcpyDeviceToDevice, s);
    if (e != cudaSuccess) return e;
    st = cb.gemm_batched(cb.handle, CUBLAS_OP_N, CUBLAS_OP_N, r, r, r, &hp.c, A, CUDA_R_32F, r, sa, A, CUDA_R_32F, r, sa,
                         &hp.b, B, CUDA_R_32F, r, sa, nb, ct, CUBLAS_GEMM_DEFAULT);
    if (st != CUBLAS_STATUS_SUCCESS) return cudaErrorUnknown;
    k_add_diag_b<<<dim3((r + 255) / 256, nb), 256, 0, s>>>(B, r, sa, hp.a);
    if (h <= w)
      st = cb.gemm_batched(cb.handle, CUBLAS_OP_N, CUBLAS_OP_N, w, h, h, &one, X, CUDA_R_32F, w, sx, B, CUDA_R_32F, r, sa,
                           &zero, X2, CUDA_R_32F, w, sx, nb, ct, CUBLAS_GEMM_DEFAULT);
    else
      st = cb.gemm_batched(cb.handle, CUBLAS_OP_N, CUBLAS_OP_N, w, h, w, &one, B, CUDA_R_32F, r, sa, X, CUDA_R_32F, w, sx,
                           &zero, X2, CUDA_R_32F, w, sx, nb, ct, CUBLAS_GEMM_DEFAULT);
    if (st != CUBLAS_STATUS_SUCCESS) return cudaErrorUnknown;
    std::swap(X, X2);
    *launches += 5;
  }
  k_update_b<S><<<grid, kEwThreads, 0, s>>>(layers_dev, items_dev, X, Th, Tw, sx, step_mode ? 1 : 0, 1.f - hp.lr * hp.wd,
                                            -hp.lr * hp.scale_c);
  *launches += 1;
  return cudaGetLastError();
}

template <typename S>
cudaError_t run_one(const LayerDev& L, const WorkItem& wi, int T, int mode, const himuon_hparams& hp, char* scratch,
                    cudaStream_t s, long long* launches) {
  Cublas& cb = cublas();
  const int row0 = (int)std::min<long long>((long long)wi.r * T, L.H), col0 = (int)std::min<long long>((long long)wi.c * T, L.W);
  const int h = (int)std::min<long long>(T, L.H - row0), w = (int)std::min<long long>(T, L.W - col0);
  if (h <= 0 || w <= 0) return cudaSuccess;
  const int r = std::min(h, w);
  const size_t xb = align256((size_t)h * w * 4), ab = align256((size_t)r * r * 4);
  float* X = reinterpret_cast<float*>(scratch);
  float* X2 = reinterpret_cast<float*>(scratch + xb);
  float* A = reinterpret_cast<float*>(scratch + 2 * xb);
  float* B = reinterpret_cast<float*>(scratch + 2 * xb + ab);
  float* partial = reinterpret_cast<float*>(scratch + 2 * xb + 2 * ab);
  void* cws = scratch + 2 * xb + 2 * ab + align256(kEwBlocks * 4);
  const bool step_mode = (mode == MODE_STEP);
  const long long n = (long long)h * w;
  const int blocks = (int)std::min<long long>(kEwBlocks, (n + kEwThreads - 1) / kEwThreads);

  View<const S> G{reinterpret_cast<const S*>(L.g) + (long long)row0 * L.ld_g + col0, L.ld_g};
  View<S> M{L.m ? reinterpret_cast<S*>(L.m) + (long long)row0 * L.ld_m + col0 : nullptr, L.ld_m};
  View<S> W{reinterpret_cast<S*>(L.w) + (long long)row0 * L.ld_w + col0, L.ld_w};

  k_prep<S><<<blocks, kEwThreads, 0, s>>>(G, M, X, partial, h, w, step_mode ? 1 : 0, hp.beta, hp.nesterov);
  k_scale<<<blocks, kEwThreads, 0, s>>>(X, partial, blocks, n, hp.eps);
  *launches += 2;

  if (hp.K > 0) {
    if (cb.set_stream(cb.handle, s) != CUBLAS_STATUS_SUCCESS) return cudaErrorUnknown;
    if (cb.set_workspace(cb.handle, cws, kCublasWs) != CUBLAS_STATUS_SUCCESS) return cudaErrorUnknown;
  }
  // fp32 storage: true fp32 products (the <= 1e-4 path); bf16 storage: TF32 tensor-core products
  const cublasComputeType_t ct = CUBLAS_COMPUTE_32F;   // this path is the true-fp32 one for either storage type
  const float one = 1.f, zero = 0.f;
  // Row-major X (h x w, ld = w) is the column-major w x h matrix Xc = X^T with leading dimension w.
  for (int k = 0; k < hp.K; ++k) {
    cublasStatus_t st;
    if (h <= w)   // A = X X^T = Xc^T Xc   (r = h)
      st = cb.gemm_ex(cb.handle, CUBLAS_OP_T, CUBLAS_OP_N, h, h, w, &one, X, CUDA_R_32F, w, X, CUDA_R_32F, w, &zero, A,
                      CUDA_R_32F, r, ct, CUBLAS_GEMM_DEFAULT);
    else          // A = X^T X = Xc Xc^T   (r = w; work on the short side)
      st = cb.gemm_ex(cb.handle, CUBLAS_OP_N, CUBLAS_OP_T, w, w, h, &one, X, CUDA_R_32F, w, X, CUDA_R_32F, w, &zero, A,
                      CUDA_R_32F, r, ct, CUBLAS_GEMM_DEFAULT);
    if (st != CUBLAS_STATUS_SUCCESS) return cudaErrorUnknown;
    cudaError_t e = cudaMemcpyAsync(B, A, (size_t)r * r * 4, cudaMemcpyDeviceToDevice, s);
    if (e != cudaSuccess) return e;
    // B = b A + c A A, then B += a I
    st = cb.gemm_ex(cb.handle, CUBLAS_OP_N, CUBLAS_OP_N, r, r, r, &hp.c, A, CUDA_R_32F, r, A, CUDA_R_32F, r, &hp.b, B,
                    CUDA_R_32F, r, ct, CUBLAS_GEMM_DEFAULT);
    if (st != CUBLAS_STATUS_SUCCESS) return cudaErrorUnknown;
    k_add_diag<<<(r + 255) / 256, 256, 0, s>>>(B, r, hp.a);
    if (h <= w)   // X <- (a I + B) X :  Xc_new = Xc (a I + B)
      st = cb.gemm_ex(cb.handle, CUBLAS_OP_N, CUBLAS_OP_N, w, h, h, &one, X, CUDA_R_32F, w, B, CUDA_R_32F, r, &zero, X2,
                      CUDA_R_32F, w, ct, CUBLAS_GEMM_DEFAULT);
    else          // X <- X (a I + B) :  Xc_new = (a I + B) Xc
      st = cb.gemm_ex(cb.handle, CUBLAS_OP_N, CUBLAS_OP_N, w, h, w, &one, B, CUDA_R_32F, r, X, CUDA_R_32F, w, &zero, X2,
                      CUDA_R_32F, w, ct, CUBLAS_GEMM_DEFAULT);
    if (st != CUBLAS_STATUS_SUCCESS) return cudaErrorUnknown;
    std::swap(X, X2);
    *launches += 5;
  }
  const float keep = 1.f - hp.lr * hp.wd;
  const float stepsz = -hp.lr * hp.scale_c * L.tau_base;
  k_update<S><<<blocks, kEwThreads, 0, s>>>(W, X, h, w, step_mode ? 1 : 0, keep, stepsz);
  *launches += 1;
  return cudaGetLastError();
}

}  // namespace

// One chunk of the work list.  Uniform tiles (T <= 512) run in sub-batches of as many tiles as the scratch holds;
// whole-matrix items run one at a time (host copies of the layer table and of the items are needed for those).
cudaError_t run_gemm_path(const LayerDev* layers_host, const WorkItem* items_host, const LayerDev* layers_dev,
                          const WorkItem* items_dev, long long n_items, int T, int Tw, int mode, int dtype,
                          const himuon_hparams& hp, void* scratch, size_t scratch_bytes, cudaStream_t s, long long* launches) {
  if (n_items < 1) return cudaSuccess;
  Cublas& cb = cublas();
  if (!cb.ok) return cudaErrorNotSupported;
  // The handle's stream and workspace are re-pointed per call: serialise the enqueueing host threads (the GPU work
  // itself stays asynchronous on each caller's stream), one handle per device.
  std::lock_guard<std::mutex> lock(cb.mu);
  if (!cb.acquire()) return cudaErrorNotSupported;
  if (T <= 2048 && Tw <= 2048 && items_dev) {
    const size_t per = gemm_path_batch_item_bytes(T, Tw);
    if (scratch_bytes < per + kCublasWs) return cudaErrorInvalidValue;
    long long cap = (long long)((scratch_bytes - kCublasWs) / per);
    if (cap > 65535) cap = 65535;   // the sub-batch index is gridDim.y of the fused ends
    for (long long i = 0; i < n_items; i += cap) {
      const int nb = (int)std::min<long long>(cap, n_items - i);
      cudaError_t e = dtype == HIMUON_F32 ? run_batch<float>(layers_dev, items_dev + i, nb, T, Tw, mode, hp, (char*)scratch, s, launches)
                                          : run_batch<__nv_bfloat16>(layers_dev, items_dev + i, nb, T, Tw, mode, hp, (char*)scratch, s, launches);
      if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
  }
  for (long long i = 0; i < n_items; ++i) {
    const WorkItem& wi = items_host[i];
    const LayerDev& L = layers_host[wi.layer];
    cudaError_t e = dtype == HIMUON_F32 ? run_one<float>(L, wi, T, mode, hp, (char*)scratch, s, launches)
                                        : run_one<__nv_bfloat16>(L, wi, T, mode, hp, (char*)scratch, s, launches);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

}  // namespace himuon
