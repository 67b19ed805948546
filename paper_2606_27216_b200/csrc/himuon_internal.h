// Internal declarations shared by the host planner, the C-ABI dispatch and the kernels.
// Not part of the public boundary (that is include/himuon.h).
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <string>
#include <vector>

#include "himuon.h"

namespace himuon {

// ---- device-visible tables (live in the caller's workspace) ---------------------------------

// One layer of the descriptor table, 64 bytes.
struct LayerDev {
  void*     w;
  void*     g;
  void*     m;
  long long ld_w, ld_g, ld_m;   // elements
  int       H, W;
  float     tau_base;           // sqrt(T) or sqrt(max(H,W)) (full branch); tau = scale_c * tau_base
  int       dtype;              // himuon_dtype
};
static_assert(sizeof(LayerDev) == 64, "LayerDev must be 64 bytes");

// One entry of the cross-layer work list: tile (r, c) of layer `layer`.
struct WorkItem {
  int layer, r, c, pad;
};
static_assert(sizeof(WorkItem) == 16, "WorkItem must be 16 bytes");

enum Mode : int { MODE_STEP = 0, MODE_PHI = 1 };
enum KernelPath : int { KPATH_FP32_SIMT = 0, KPATH_TC = 1, KPATH_WARP = 2, KPATH_GEMM = 3, KPATH_TC_FP8 = 4, KPATH_LT = 5 };
inline bool kpath_uses_tma(int kp) { return kp == KPATH_TC || kp == KPATH_TC_FP8; }
constexpr int kWholeMatrixT = 1 << 20;   // tile size of the full-matrix branch beyond the largest tile kernel (R = C = 1)

struct LaunchArgs {
  const LayerDev*    layers;     // device
  const CUtensorMap* tmaps;      // device, 3 per layer (w, g, m); may be null on the SIMT path
  const WorkItem*    items;      // device; null => implicit list: item i = (layer 0, r = i, c = 0)
  long long          n_items;
  int                T;
  int                mode;
  int                dtype;      // storage dtype of every layer in this launch (bucket key)
  himuon_hparams     hp;
};

// kernels_simt.cu -- fp32 FMA path, T in {16, 32, 64, 128}, fp32 or bf16 storage.
cudaError_t launch_simt(const LaunchArgs& a, cudaStream_t stream);
// kernels_tc128.cu -- tcgen05 bf16 path, T = 128, bf16 storage.
cudaError_t launch_tc128(const LaunchArgs& a, cudaStream_t stream);
cudaError_t launch_tc128_fp8(const LaunchArgs& a, cudaStream_t stream);   // e4m3 operands, HIMUON_PATH_FP8
cudaError_t launch_tc256_fp8(const LaunchArgs& a, cudaStream_t stream);
// kernels_tc64.cu -- tcgen05 bf16 path, T = 64 (two tiles stacked per MMA), bf16 storage.
cudaError_t launch_tc64(const LaunchArgs& a, cudaStream_t stream);
// kernels_tc256.cu -- tcgen05 cta_group::2 bf16 path, T = 256 (one tile per CTA pair), bf16 storage.
cudaError_t launch_tc256(const LaunchArgs& a, cudaStream_t stream);
// kernels_warp.cu -- mma.sync bf16 path, one warp per tile, T in {16, 32}, bf16 storage.
cudaError_t launch_warp(const LaunchArgs& a, cudaStream_t stream);

// kernels_gemm.cu -- large tiles in TRUE fp32 arithmetic (fp32 storage, HIMUON_PATH_FP32): fp32 cuBLAS products, host walk.
size_t      gemm_path_scratch_bytes(int h, int w);        // one whole h x w block at a time
size_t      gemm_path_batch_item_bytes(int Th, int Tw);   // per tile of a sub-batch of uniform Th x Tw tiles
size_t      gemm_path_fixed_bytes();                      // cuBLAS workspace inside the scratch
cudaError_t run_gemm_path(const LayerDev* layers_host, const WorkItem* items_host, const LayerDev* layers_dev,
                          const WorkItem* items_dev, long long n_items, int T, int Tw, int mode, int dtype,
                          const himuon_hparams& hp, void* scratch, size_t scratch_bytes, cudaStream_t stream,
                          long long* launches);

// SM count of the CURRENT device (per-device cache, thread-safe).
// kernels_lt.cu -- large tiles on bf16 storage (T = 512, full-matrix branch beyond 256, rectangular tiles): hand-written
// persistent tcgen05 GEMMs with the Newton-Schulz step fused into their epilogues, one launch per product per sub-batch.
size_t      lt_path_scratch_bytes(int h, int w);          // one whole h x w block
size_t      lt_path_batch_item_bytes(int Th, int Tw);     // per tile of a sub-batch of uniform Th x Tw tiles
cudaError_t run_lt_path(const LayerDev* layers_host, const WorkItem* items_host, const LayerDev* layers_dev,
                        const WorkItem* items_dev, long long n_items, int T, int Tw, int mode, const himuon_hparams& hp,
                        void* scratch, size_t scratch_bytes, cudaStream_t stream, long long* launches);

int device_sm_count();

// One-time kernel configuration (dynamic shared memory size) per DEVICE: `done` holds one bit per device
// ordinal.  Thread-safe: two threads racing on the same device both set the (idempotent) attribute.
struct DeviceOnce {
  std::atomic<unsigned long long> done{0};
};
template <typename Kernel>
cudaError_t configure_smem_once(DeviceOnce& once, Kernel kernel, int smem_bytes) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  const unsigned long long bit = 1ull << (dev & 63);
  if (dev < 64 && (once.done.load(std::memory_order_acquire) & bit)) return cudaSuccess;
  e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
  if (e != cudaSuccess) return e;
  if (dev < 64) once.done.fetch_or(bit, std::memory_order_release);
  return cudaSuccess;
}

// ---- host plan --------------------------------------------------------------------------------

struct Bucket {
  int       T;            // tile rows
  int       Tw;           // tile columns (= T except for rectangular tiles)
  int       dtype;
  int       kpath;
  long long begin, end;   // range in the work list
};

struct Chunk {
  int       bucket;
  long long begin, end;
};

}  // namespace himuon

struct himuon_plan {
  std::vector<himuon_layer>     layers;
  std::vector<int>              T_eff;       // per layer, effective (supported) tile size (rows)
  std::vector<int>              Tw_eff;      // per layer, tile columns (= T_eff except for rectangular tiles)
  std::vector<int>              kpath;       // per layer
  std::vector<himuon::LayerDev> layer_dev;
  std::vector<himuon::WorkItem> items;       // execution order
  std::vector<himuon::Bucket>   buckets;
  std::vector<himuon::Chunk>    chunks;
  bool      resident  = true;                // whole list fits under the cap
  bool      bindable  = true;                // all pointers non-null
  bool      needs_tma = false;
  size_t    fixed_bytes = 0;                 // layer table + tensor maps
  size_t    off_tmaps = 0, off_items = 0, off_scratch = 0;
  size_t    scratch_bytes = 0;               // large-tile path only
  long long max_chunk_tiles = 0;
  size_t    workspace_bytes = 0;
  size_t    cap = 0;
  // binding
  void*             ws = nullptr;
  himuon::WorkItem* pinned_items = nullptr;  // streaming mode only
};
