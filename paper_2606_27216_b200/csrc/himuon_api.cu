// C-ABI of the HiMuon hot path: host planner (cross-layer work list, buckets, memory-bounded
// chunking -- PAPER.md:231-241, sec. 4.4.2-4.4.3), binding of the plan's device tables, and dispatch
// of one kernel launch per chunk.  See include/himuon.h for the contract of every entry point.
#include <atomic>
#include <map>
#include <mutex>
#include <string>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "himuon_internal.h"

using namespace himuon;

namespace {

thread_local std::string g_last_cuda_error;
std::atomic<long long>   g_launches{0};

himuon_status cuda_fail(cudaError_t e, const char* what) {
  g_last_cuda_error = std::string(what) + ": " + cudaGetErrorString(e);
  return HIMUON_ERR_CUDA;
}

constexpr size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

const int kTileSizes[] = {16, 32, 64, 128, 256, 512};

// Which kernel serves (dtype, requested path, T); -1 = none in this build.
// W = number of columns of the matrix (0 = unknown / any).  The TMA stores of the tensor-core path
// work in 16-byte granules of a row, so a bf16 matrix whose width is not a multiple of 8 is served
// by the fp32 kernel instead (measured on B200: a store clipped at such a width zero-fills the rest
// of the last granule, i.e. it would write into the ld - W gutter).
int select_kpath(int dtype, int path, int T, int W = 0) {
  const bool simt_ok = (T == 16 || T == 32 || T == 64 || T == 128);
  if (path == HIMUON_PATH_FP8)                                      // e4m3 operands: the T = 128 / 256 tcgen05 kernels only
    return (dtype == HIMUON_BF16 && (T == 128 || T == 256) && (W % 8) == 0) ? KPATH_TC_FP8 : -1;
  // true fp32 arithmetic (the <= 1e-4 path): FMA kernel up to T = 128, fp32 cuBLAS products beyond
  if (path == HIMUON_PATH_FP32 || dtype == HIMUON_F32) return simt_ok ? KPATH_FP32_SIMT : (T >= 256 ? KPATH_GEMM : -1);
  // bf16 storage, AUTO: tensor-core kernels; large tiles: the tcgen05 GEMM path with fused epilogues.
  if (T >= 512) return KPATH_LT;
  if ((T == 256 || T == 128 || T == 64) && (W % 8) == 0) return KPATH_TC;
  if (T == 16 || T == 32) return KPATH_WARP;
  if (T == 256) return KPATH_LT;                                    // width not a multiple of 8
  return simt_ok ? KPATH_FP32_SIMT : -1;
}

int smallest_supported_T_at_least(int n, int dtype, int path) {
  for (int T : kTileSizes)
    if (T >= n && select_kpath(dtype, path, T) >= 0) return T;
  return -1;
}

bool valid_hparams(const himuon_hparams* hp) {
  if (!hp) return false;
  if (hp->K < 0 || hp->K > 64) return false;
  if (!(hp->eps >= 0.f)) return false;
  if (!std::isfinite(hp->a) || !std::isfinite(hp->b) || !std::isfinite(hp->c)) return false;
  if (!std::isfinite(hp->beta) || !std::isfinite(hp->lr) || !std::isfinite(hp->wd) ||
      !std::isfinite(hp->scale_c))
    return false;
  return true;
}

// The tcgen05 kernels (tc64, tc128, tc256, their e4m3 variants and the large-tile GEMM path) iterate on the scaled state
// c^(1/4) X with beta = b / sqrt(c), which needs c > 0.  The fp32 kernels and the warp kernel
// (T = 16, 32: plain state, polynomial in fp32) take any finite (a, b, c), e.g. the cubic iteration (1.5, -0.5, 0).
bool kpath_needs_positive_c(int kp) { return kp == KPATH_TC || kp == KPATH_TC_FP8 || kp == KPATH_LT; }
bool positive_c_ok(const himuon_hparams* hp) {
  return hp->c > 0.f && std::isfinite(hp->b / std::sqrt(hp->c)) && std::isfinite(1.f / std::sqrt(std::sqrt(hp->c)));
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static bool          tried = false;
  if (!tried) {
    tried = true;
    void*                            p = nullptr;
    cudaDriverEntryPointQueryResult  q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

// bf16 row-major H x W matrix with leading dimension ld; box = 64 columns (128 B, one swizzle
// span) x box_rows rows; out-of-bounds elements read as zero and are clipped on store, which is
// exactly the zero padding / cropping of B_T and B_T^-1.
bool encode_bf16_map(CUtensorMap* out, void* ptr, int H, int W, long long ld, int box_rows) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2]    = {(cuuint64_t)W, (cuuint64_t)H};
  cuuint64_t strides[1] = {(cuuint64_t)ld * 2};
  cuuint32_t box[2]     = {64u, (cuuint32_t)box_rows};
  cuuint32_t estr[2]    = {1u, 1u};
  CUresult   r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, ptr, dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

// e4m3 operands need enough singular directions to average their rounding over: an edge tile with fewer than
// kFp8MinLive live rows or columns (e.g. a 44 x 8 corner block, measured 0.19 against the path's 0.15 bound) is run
// by the bf16 kernel of the same tile size instead - its own bucket of the same plan (buckets are
// keyed by kernel path).  DESIGN.md section 5.
constexpr int kFp8MinLive = 32;
int tile_kpath(int layer_kpath, int H, int W, int T, int Tw, int r, int c) {
  if (layer_kpath != KPATH_TC_FP8) return layer_kpath;
  const int lh = H - r * T < T ? H - r * T : T, lw = W - c * Tw < Tw ? W - c * Tw : Tw;
  return (lh < kFp8MinLive || lw < kFp8MinLive) ? KPATH_TC : KPATH_TC_FP8;
}

himuon_status chunk_rule(long long n_items, long long bytes_per_item, long long fixed_bytes,
                         long long cap_bytes, std::vector<long long>& offs) {
  offs.clear();
  offs.push_back(0);
  if (n_items < 0 || bytes_per_item < 0 || fixed_bytes < 0) return HIMUON_ERR_INVALID_ARG;
  if (n_items == 0) return HIMUON_OK;
  long long per_chunk_max;
  if (cap_bytes <= 0 || bytes_per_item == 0) {
    per_chunk_max = n_items;
  } else {
    per_chunk_max = (cap_bytes - fixed_bytes) / bytes_per_item;
    if (cap_bytes < fixed_bytes || per_chunk_max < 1) return HIMUON_ERR_WORKSPACE_TOO_SMALL;
    if (per_chunk_max > n_items) per_chunk_max = n_items;
  }
  long long n_chunks = (n_items + per_chunk_max - 1) / per_chunk_max;
  long long base = n_items / n_chunks, rem = n_items % n_chunks;
  for (long long i = 0; i < n_chunks; ++i) offs.push_back(offs.back() + base + (i < rem ? 1 : 0));
  return HIMUON_OK;
}

cudaError_t launch_chunk(const LaunchArgs& a, int kpath, cudaStream_t s) {
  g_launches.fetch_add(1);
  if (kpath == KPATH_TC_FP8) return a.T == 256 ? launch_tc256_fp8(a, s) : launch_tc128_fp8(a, s);
  if (kpath == KPATH_TC) return a.T == 64 ? launch_tc64(a, s) : a.T == 256 ? launch_tc256(a, s) : launch_tc128(a, s);
  if (kpath == KPATH_WARP) return launch_warp(a, s);
  return launch_simt(a, s);
}

}  // namespace

namespace himuon {
int device_sm_count() {
  static std::atomic<int> cache[64];   // zero-initialised; one entry per device ordinal
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 148;
  if (dev >= 0 && dev < 64) {
    const int c = cache[dev].load(std::memory_order_relaxed);
    if (c > 0) return c;
  }
  int n = 0;
  if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return 148;
  if (dev >= 0 && dev < 64) cache[dev].store(n, std::memory_order_relaxed);
  return n;
}
}  // namespace himuon

extern "C" {

const char* himuon_status_string(himuon_status s) {
  switch (s) {
    case HIMUON_OK: return "HIMUON_OK";
    case HIMUON_ERR_INVALID_ARG: return "HIMUON_ERR_INVALID_ARG";
    case HIMUON_ERR_UNSUPPORTED: return "HIMUON_ERR_UNSUPPORTED";
    case HIMUON_ERR_WORKSPACE_TOO_SMALL: return "HIMUON_ERR_WORKSPACE_TOO_SMALL";
    case HIMUON_ERR_CUDA: return "HIMUON_ERR_CUDA";
    case HIMUON_ERR_NOT_BOUND: return "HIMUON_ERR_NOT_BOUND";
  }
  return "HIMUON_ERR_UNKNOWN";
}

const char* himuon_last_cuda_error(void) { return g_last_cuda_error.c_str(); }

int64_t himuon_launch_count(void) { return g_launches.load(); }

int32_t himuon_supported_tile_sizes(int32_t dtype, int32_t path) {
  int32_t mask = 0;
  for (int i = 0; i < (int)(sizeof(kTileSizes) / sizeof(kTileSizes[0])); ++i)
    if (select_kpath(dtype, path, kTileSizes[i]) >= 0) mask |= (1 << i);
  return mask;
}

himuon_status himuon_plan_chunks(int64_t n_items, int64_t bytes_per_item, int64_t fixed_bytes,
                                 int64_t cap_bytes, int32_t* n_chunks, int64_t* offsets_out,
                                 int32_t offsets_capacity) {
  if (!n_chunks) return HIMUON_ERR_INVALID_ARG;
  std::vector<long long> offs;
  himuon_status st = chunk_rule(n_items, bytes_per_item, fixed_bytes, cap_bytes, offs);
  if (st != HIMUON_OK) return st;
  *n_chunks = (int32_t)offs.size() - 1;
  if (offsets_out) {
    if (offsets_capacity < (int32_t)offs.size()) return HIMUON_ERR_INVALID_ARG;
    for (size_t i = 0; i < offs.size(); ++i) offsets_out[i] = offs[i];
  }
  return HIMUON_OK;
}

himuon_status himuon_plan_create(const himuon_layer* layers, int32_t n_layers, int32_t T_default,
                                 int32_t path, size_t workspace_cap_bytes, himuon_plan** out) {
  if (!out) return HIMUON_ERR_INVALID_ARG;
  *out = nullptr;
  if (!layers || n_layers <= 0) return HIMUON_ERR_INVALID_ARG;
  if (path != HIMUON_PATH_AUTO && path != HIMUON_PATH_FP32 && path != HIMUON_PATH_FP8) return HIMUON_ERR_INVALID_ARG;
  if (T_default < 0) return HIMUON_ERR_INVALID_ARG;

  himuon_plan* p = new (std::nothrow) himuon_plan();
  if (!p) return HIMUON_ERR_INVALID_ARG;
  p->cap = workspace_cap_bytes;
  p->layers.assign(layers, layers + n_layers);
  p->T_eff.resize(n_layers);
  p->Tw_eff.resize(n_layers);
  p->kpath.resize(n_layers);
  p->layer_dev.resize(n_layers);

  himuon_status st = HIMUON_OK;
  std::map<int, long long> gemm_tiles;   // large-tile path: tiles per tile size so far
  for (int l = 0; l < n_layers && st == HIMUON_OK; ++l) {
    const himuon_layer& L = layers[l];
    const int H = L.g.H, W = L.g.W, dt = L.g.dtype;
    if (H <= 0 || W <= 0 || (dt != HIMUON_F32 && dt != HIMUON_BF16)) { st = HIMUON_ERR_INVALID_ARG; break; }
    if (L.w.H != H || L.w.W != W || L.w.dtype != dt) { st = HIMUON_ERR_INVALID_ARG; break; }
    if (L.m.ptr && (L.m.H != H || L.m.W != W || L.m.dtype != dt)) { st = HIMUON_ERR_INVALID_ARG; break; }
    if (L.g.ld < W || L.w.ld < W || (L.m.ptr && L.m.ld < W)) { st = HIMUON_ERR_INVALID_ARG; break; }
    int T = L.T > 0 ? L.T : T_default;
    if (T <= 0 || L.T < 0 || L.T_w < 0) { st = HIMUON_ERR_INVALID_ARG; break; }
    const int  mx = H > W ? H : W;
    const bool rect = L.T_w > 0 && L.T_w != T && !(T >= H && L.T_w >= W);   // rectangular tiles
    const bool full = rect ? false : (L.T_w > 0 && L.T_w != T ? true : T >= mx);   // full-matrix branch
    int Te, Twe = 0;
    if (rect) {
      auto pow2_ok = [](int v) { return v >= 16 && v <= 2048 && (v & (v - 1)) == 0; };
      if (!pow2_ok(T) || !pow2_ok(L.T_w)) { st = HIMUON_ERR_INVALID_ARG; break; }
      Te = T;
      Twe = L.T_w;
    } else if (full) {
      Te = smallest_supported_T_at_least(mx, dt, path);
      if (Te < 0) Te = kWholeMatrixT;          // larger than every tile size: one whole-matrix item on the cuBLAS path
    } else {
      bool known = false;
      for (int t : kTileSizes) known |= (t == T);
      if (!known) { st = HIMUON_ERR_INVALID_ARG; break; }
      if (select_kpath(dt, path, T) < 0) { st = HIMUON_ERR_UNSUPPORTED; break; }
      Te = T;
    }
    if (rect && path == HIMUON_PATH_FP8) { st = HIMUON_ERR_UNSUPPORTED; break; }   // e4m3 operands: square tiles only
    const int kp = rect ? ((dt == HIMUON_BF16 && path == HIMUON_PATH_AUTO) ? KPATH_LT : KPATH_GEMM) : select_kpath(dt, path, Te, W);
    if (kp < 0) { st = HIMUON_ERR_UNSUPPORTED; break; }
    if (!rect) Twe = Te;
    if (kp == KPATH_GEMM || kp == KPATH_LT) {
      const bool lt = (kp == KPATH_LT);
      size_t need;
      if (Te <= 2048 && Twe <= 2048) {   // uniform tiles run in sub-batches: as many tiles as a scratch budget holds (>= 1)
        const size_t per = lt ? lt_path_batch_item_bytes(Te, Twe) : gemm_path_batch_item_bytes(Te, Twe);
        size_t       budget = (size_t)1024 << 20;
        if (workspace_cap_bytes && workspace_cap_bytes / 2 < budget) budget = workspace_cap_bytes / 2;
        const int key = (Te * 4096 + Twe) * 2 + (lt ? 1 : 0);
        gemm_tiles[key] += (long long)((H + Te - 1) / Te) * ((W + Twe - 1) / Twe);
        long long nb = (long long)(budget / per);
        if (nb > gemm_tiles[key]) nb = gemm_tiles[key];
        if (nb < 1) nb = 1;
        need = (lt ? 0 : gemm_path_fixed_bytes()) + (size_t)nb * per;
      } else {
        need = lt ? lt_path_scratch_bytes(H, W) : gemm_path_scratch_bytes(H, W);
      }
      if (need > p->scratch_bytes) p->scratch_bytes = need;
    }
    p->T_eff[l] = Te;
    p->Tw_eff[l] = Twe;
    p->kpath[l] = kp;
    if (!L.g.ptr || !L.w.ptr) p->bindable = false;
    const size_t esz = dt == HIMUON_BF16 ? 2 : 4;
    if (kpath_uses_tma(kp)) {
      p->needs_tma = true;
      const himuon_mat* ms[3] = {&L.w, &L.g, &L.m};
      for (int i = 0; i < 3; ++i) {
        if (!ms[i]->ptr) continue;
        if (((uintptr_t)ms[i]->ptr & 15) || ((ms[i]->ld * (long long)esz) & 15)) { st = HIMUON_ERR_UNSUPPORTED; break; }
      }
    } else {
      const himuon_mat* ms[3] = {&L.w, &L.g, &L.m};
      for (int i = 0; i < 3; ++i)
        if (ms[i]->ptr && ((uintptr_t)ms[i]->ptr & (esz - 1))) st = HIMUON_ERR_INVALID_ARG;
    }
    LayerDev& D = p->layer_dev[l];
    D.w = L.w.ptr; D.g = L.g.ptr; D.m = L.m.ptr;
    D.ld_w = L.w.ld; D.ld_g = L.g.ld; D.ld_m = L.m.ptr ? L.m.ld : 0;
    D.H = H; D.W = W; D.dtype = dt;
    D.tau_base = std::sqrt((float)(full ? mx : (rect ? (T > L.T_w ? T : L.T_w) : T)));
  }
  if (st != HIMUON_OK) { delete p; return st; }

  // Buckets in order of first appearance; work list = bucket-major, then layer order, then r-major.
  for (int l = 0; l < n_layers; ++l) {
    int dt = layers[l].g.dtype, bi = -1;
    for (size_t b = 0; b < p->buckets.size(); ++b)
      if (p->buckets[b].T == p->T_eff[l] && p->buckets[b].Tw == p->Tw_eff[l] && p->buckets[b].dtype == dt &&
          p->buckets[b].kpath == p->kpath[l])
        bi = (int)b;
    if (bi < 0) p->buckets.push_back(Bucket{p->T_eff[l], p->Tw_eff[l], dt, p->kpath[l], 0, 0});
    if (p->kpath[l] == KPATH_TC_FP8) {   // small edge tiles of an e4m3 layer: companion bf16 bucket
      const int T = p->T_eff[l], H = layers[l].g.H, W = layers[l].g.W;
      const bool small = (H % T != 0 && H % T < kFp8MinLive) || (W % T != 0 && W % T < kFp8MinLive);
      bool have = false;
      for (const Bucket& B : p->buckets) have |= (B.T == T && B.Tw == T && B.dtype == dt && B.kpath == KPATH_TC);
      if (small && !have) p->buckets.push_back(Bucket{T, T, dt, KPATH_TC, 0, 0});
    }
  }
  for (size_t b = 0; b < p->buckets.size(); ++b) {
    Bucket& B = p->buckets[b];
    B.begin = (long long)p->items.size();
    for (int l = 0; l < n_layers; ++l) {
      if (p->T_eff[l] != B.T || p->Tw_eff[l] != B.Tw || layers[l].g.dtype != B.dtype) continue;
      if (p->kpath[l] != B.kpath && !(p->kpath[l] == KPATH_TC_FP8 && B.kpath == KPATH_TC)) continue;
      const int H = layers[l].g.H, W = layers[l].g.W;
      const int R = (H + B.T - 1) / B.T, C = (W + B.Tw - 1) / B.Tw;
      for (int r = 0; r < R; ++r)
        for (int c = 0; c < C; ++c)
          if (tile_kpath(p->kpath[l], H, W, B.T, B.Tw, r, c) == B.kpath) p->items.push_back(WorkItem{l, r, c, 0});
    }
    B.end = (long long)p->items.size();
  }

  // Workspace layout: [layer table][tensor maps][work items of the resident list / current chunk].
  p->off_tmaps   = align_up((size_t)n_layers * sizeof(LayerDev), 128);
  p->off_scratch = align_up(p->off_tmaps + (p->needs_tma ? (size_t)n_layers * 3 * sizeof(CUtensorMap) : 0), 256);
  p->off_items   = p->off_scratch + p->scratch_bytes;
  p->fixed_bytes = p->off_items;
  const long long n_total = (long long)p->items.size();
  std::vector<long long> offs;
  st = chunk_rule(n_total, sizeof(WorkItem), (long long)p->fixed_bytes, (long long)workspace_cap_bytes, offs);
  if (st != HIMUON_OK) { delete p; return st; }
  p->resident = (offs.size() <= 2);
  if (p->resident) {
    for (size_t b = 0; b < p->buckets.size(); ++b)
      p->chunks.push_back(Chunk{(int)b, p->buckets[b].begin, p->buckets[b].end});
    p->max_chunk_tiles = n_total;
  } else {
    for (size_t b = 0; b < p->buckets.size(); ++b) {
      const Bucket& B = p->buckets[b];
      std::vector<long long> bo;
      st = chunk_rule(B.end - B.begin, sizeof(WorkItem), (long long)p->fixed_bytes, (long long)workspace_cap_bytes, bo);
      if (st != HIMUON_OK) { delete p; return st; }
      for (size_t i = 0; i + 1 < bo.size(); ++i) {
        p->chunks.push_back(Chunk{(int)b, B.begin + bo[i], B.begin + bo[i + 1]});
        if (bo[i + 1] - bo[i] > p->max_chunk_tiles) p->max_chunk_tiles = bo[i + 1] - bo[i];
      }
    }
  }
  p->workspace_bytes = p->fixed_bytes + (size_t)p->max_chunk_tiles * sizeof(WorkItem);
  if (p->workspace_bytes < 128) p->workspace_bytes = 128;
  *out = p;
  return HIMUON_OK;
}

himuon_status himuon_plan_info(const himuon_plan* plan, int64_t* n_tiles, int32_t* n_buckets,
                               int32_t* n_chunks, size_t* workspace_bytes) {
  if (!plan) return HIMUON_ERR_INVALID_ARG;
  if (n_tiles) *n_tiles = (int64_t)plan->items.size();
  if (n_buckets) *n_buckets = (int32_t)plan->buckets.size();
  if (n_chunks) *n_chunks = (int32_t)plan->chunks.size();
  if (workspace_bytes) *workspace_bytes = plan->workspace_bytes;
  return HIMUON_OK;
}

himuon_status himuon_plan_worklist(const himuon_plan* plan, int32_t* lrc_out, int64_t* chunk_offsets,
                                   int32_t* bucket_T_out) {
  if (!plan) return HIMUON_ERR_INVALID_ARG;
  if (lrc_out)
    for (size_t i = 0; i < plan->items.size(); ++i) {
      lrc_out[3 * i + 0] = plan->items[i].layer;
      lrc_out[3 * i + 1] = plan->items[i].r;
      lrc_out[3 * i + 2] = plan->items[i].c;
    }
  if (chunk_offsets) {
    for (size_t i = 0; i < plan->chunks.size(); ++i) chunk_offsets[i] = plan->chunks[i].begin;
    chunk_offsets[plan->chunks.size()] = (int64_t)plan->items.size();
  }
  if (bucket_T_out)
    for (size_t i = 0; i < plan->chunks.size(); ++i) bucket_T_out[i] = plan->buckets[plan->chunks[i].bucket].T;
  return HIMUON_OK;
}

void himuon_plan_destroy(himuon_plan* plan) {
  if (!plan) return;
  if (plan->pinned_items) cudaFreeHost(plan->pinned_items);
  delete plan;
}

himuon_status himuon_plan_bind(himuon_plan* plan, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!plan || !workspace) return HIMUON_ERR_INVALID_ARG;
  if (!plan->bindable) return HIMUON_ERR_INVALID_ARG;
  if (workspace_bytes < plan->workspace_bytes) return HIMUON_ERR_WORKSPACE_TOO_SMALL;
  if ((uintptr_t)workspace & 127) return HIMUON_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  char*        ws = (char*)workspace;
  const int    n = (int)plan->layers.size();
  cudaError_t  e = cudaMemcpyAsync(ws, plan->layer_dev.data(), (size_t)n * sizeof(LayerDev), cudaMemcpyHostToDevice, s);
  if (e != cudaSuccess) return cuda_fail(e, "bind: layer table");
  if (plan->needs_tma) {
    std::vector<CUtensorMap> maps((size_t)n * 3);
    std::memset(maps.data(), 0, maps.size() * sizeof(CUtensorMap));
    for (int l = 0; l < n; ++l) {
      if (!kpath_uses_tma(plan->kpath[l])) continue;
      const himuon_layer& L = plan->layers[l];
      const himuon_mat*   ms[3] = {&L.w, &L.g, &L.m};
      for (int i = 0; i < 3; ++i) {
        if (!ms[i]->ptr) continue;
        if (!encode_bf16_map(&maps[(size_t)l * 3 + i], ms[i]->ptr, ms[i]->H, ms[i]->W, ms[i]->ld, plan->T_eff[l] > 128 ? 128 : plan->T_eff[l])) {
          g_last_cuda_error = "bind: cuTensorMapEncodeTiled failed or unavailable";
          return HIMUON_ERR_CUDA;
        }
      }
    }
    e = cudaMemcpyAsync(ws + plan->off_tmaps, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return cuda_fail(e, "bind: tensor maps");
    // pageable source: the runtime has staged the bytes when the call returns.
  }
  if (plan->resident) {
    if (!plan->items.empty()) {
      e = cudaMemcpyAsync(ws + plan->off_items, plan->items.data(), plan->items.size() * sizeof(WorkItem),
                          cudaMemcpyHostToDevice, s);
      if (e != cudaSuccess) return cuda_fail(e, "bind: work list");
    }
  } else if (!plan->pinned_items) {
    e = cudaHostAlloc((void**)&plan->pinned_items, plan->items.size() * sizeof(WorkItem), cudaHostAllocDefault);
    if (e != cudaSuccess) return cuda_fail(e, "bind: pinned work list");
    std::memcpy(plan->pinned_items, plan->items.data(), plan->items.size() * sizeof(WorkItem));
  }
  plan->ws = workspace;
  return HIMUON_OK;
}

static himuon_status run_plan(himuon_plan* plan, const himuon_hparams* hp, int mode, void* cuda_stream) {
  if (!plan || !valid_hparams(hp)) return HIMUON_ERR_INVALID_ARG;
  for (const Bucket& B : plan->buckets)          // before any launch (and before the bound check: pure argument validation)
    if (B.end > B.begin && kpath_needs_positive_c(B.kpath) && !positive_c_ok(hp)) return HIMUON_ERR_UNSUPPORTED;
  if (!plan->ws) return HIMUON_ERR_NOT_BOUND;
  if (mode == MODE_STEP)
    for (const himuon_layer& L : plan->layers)
      if (!L.m.ptr) return HIMUON_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  char*        ws = (char*)plan->ws;
  for (const Chunk& c : plan->chunks) {
    if (c.end == c.begin) continue;
    const Bucket& B = plan->buckets[c.bucket];
    LaunchArgs    a;
    a.layers = (const LayerDev*)ws;
    a.tmaps  = plan->needs_tma ? (const CUtensorMap*)(ws + plan->off_tmaps) : nullptr;
    if (plan->resident) {
      a.items = (const WorkItem*)(ws + plan->off_items) + c.begin;
    } else {
      cudaError_t e = cudaMemcpyAsync(ws + plan->off_items, plan->pinned_items + c.begin,
                                      (size_t)(c.end - c.begin) * sizeof(WorkItem), cudaMemcpyHostToDevice, s);
      if (e != cudaSuccess) return cuda_fail(e, "step: chunk work list");
      a.items = (const WorkItem*)(ws + plan->off_items);
    }
    if (B.kpath == KPATH_LT) {     // large tiles, bf16: tcgen05 GEMMs with fused epilogues (sub-batches of tiles / whole matrices)
      long long   n_launch = 0;
      cudaError_t e = run_lt_path(plan->layer_dev.data(), plan->items.data() + c.begin, a.layers, a.items, c.end - c.begin,
                                  B.T, B.Tw, mode, *hp, ws + plan->off_scratch, plan->scratch_bytes, s, &n_launch);
      g_launches.fetch_add(n_launch);
      if (e != cudaSuccess) return cuda_fail(e, "step: large-tile path");
      continue;
    }
    if (B.kpath == KPATH_GEMM) {   // large tiles in true fp32: products go to cuBLAS (sub-batches of tiles / whole matrices)
      long long   n_launch = 0;
      cudaError_t e = run_gemm_path(plan->layer_dev.data(), plan->items.data() + c.begin, a.layers, a.items,
                                    c.end - c.begin, B.T, B.Tw, mode, B.dtype, *hp, ws + plan->off_scratch,
                                    plan->scratch_bytes, s, &n_launch);
      g_launches.fetch_add(n_launch);
      if (e != cudaSuccess) return cuda_fail(e, "step: large-tile path (cuBLAS)");
      continue;
    }
    a.n_items = c.end - c.begin;
    a.T = B.T;
    a.mode = mode;
    a.dtype = B.dtype;
    a.hp = *hp;
    cudaError_t e = launch_chunk(a, B.kpath, s);
    if (e != cudaSuccess) return cuda_fail(e, "step: kernel launch");
  }
  return HIMUON_OK;
}

himuon_status himuon_step(himuon_plan* plan, const himuon_hparams* hp, void* cuda_stream) {
  return run_plan(plan, hp, MODE_STEP, cuda_stream);
}

himuon_status himuon_phi(himuon_plan* plan, const himuon_hparams* hp, void* cuda_stream) {
  return run_plan(plan, hp, MODE_PHI, cuda_stream);
}

static size_t ns_tiles_scratch_bytes() {   // fp32 cuBLAS path: one 512-tile; tcgen05 large-tile path: sub-batches of 32
  const size_t a = gemm_path_scratch_bytes(512, 512), b = 32 * lt_path_batch_item_bytes(512, 512);
  return a > b ? a : b;
}
size_t himuon_ns_tiles_workspace_bytes(void) {
  return align_up(128 + 3 * sizeof(CUtensorMap), 256) + ns_tiles_scratch_bytes();
}

himuon_status himuon_ns_tiles(const void* tiles_in, void* tiles_out, int64_t n_tiles, int32_t T,
                              int32_t dtype, int32_t path, int32_t K, float a, float b, float c,
                              float eps, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (n_tiles < 0) return HIMUON_ERR_INVALID_ARG;
  if (dtype != HIMUON_F32 && dtype != HIMUON_BF16) return HIMUON_ERR_INVALID_ARG;
  if (path != HIMUON_PATH_AUTO && path != HIMUON_PATH_FP32 && path != HIMUON_PATH_FP8) return HIMUON_ERR_INVALID_ARG;
  bool known = false;
  for (int t : kTileSizes) known |= (t == T);
  if (!known) return HIMUON_ERR_INVALID_ARG;
  himuon_hparams hp;
  std::memset(&hp, 0, sizeof(hp));
  hp.K = K; hp.a = a; hp.b = b; hp.c = c; hp.eps = eps;
  if (!valid_hparams(&hp)) return HIMUON_ERR_INVALID_ARG;
  const int kp = select_kpath(dtype, path, T);
  if (kp < 0) return HIMUON_ERR_UNSUPPORTED;
  if (kpath_needs_positive_c(kp) && !positive_c_ok(&hp)) return HIMUON_ERR_UNSUPPORTED;
  if (n_tiles == 0) return HIMUON_OK;
  if (!tiles_in || !tiles_out || !workspace) return HIMUON_ERR_INVALID_ARG;
  if (n_tiles * (int64_t)T > 0x7fffffffLL) return HIMUON_ERR_UNSUPPORTED;
  if (workspace_bytes < himuon_ns_tiles_workspace_bytes()) return HIMUON_ERR_WORKSPACE_TOO_SMALL;
  if ((uintptr_t)workspace & 127) return HIMUON_ERR_INVALID_ARG;
  const size_t esz = dtype == HIMUON_BF16 ? 2 : 4;
  if (kpath_uses_tma(kp) && (((uintptr_t)tiles_in & 15) || ((uintptr_t)tiles_out & 15))) return HIMUON_ERR_UNSUPPORTED;
  if (((uintptr_t)tiles_in & (esz - 1)) || ((uintptr_t)tiles_out & (esz - 1))) return HIMUON_ERR_INVALID_ARG;

  // The packed batch is one (n_tiles*T) x T matrix whose tile (r, 0) is tile r.
  cudaStream_t s = (cudaStream_t)cuda_stream;
  char*        ws = (char*)workspace;
  LayerDev     D;
  D.w = tiles_out; D.g = const_cast<void*>(tiles_in); D.m = nullptr;
  D.ld_w = T; D.ld_g = T; D.ld_m = 0;
  D.H = (int)(n_tiles * T); D.W = T; D.tau_base = 0.f; D.dtype = dtype;
  if (kp == KPATH_LT) {     // large tiles, bf16: tcgen05 GEMM path over the implicit list of the packed batch
    long long   n_launch = 0;
    cudaError_t el = cudaMemcpyAsync(ws, &D, sizeof(D), cudaMemcpyHostToDevice, s);
    if (el != cudaSuccess) return cuda_fail(el, "ns_tiles: layer table");
    el = run_lt_path(&D, nullptr, (const LayerDev*)ws, nullptr, n_tiles, T, T, MODE_PHI, hp,
                     ws + align_up(128 + 3 * sizeof(CUtensorMap), 256), ns_tiles_scratch_bytes(), s, &n_launch);
    g_launches.fetch_add(n_launch);
    if (el != cudaSuccess) return cuda_fail(el, "ns_tiles: large-tile path");
    return HIMUON_OK;
  }
  if (kp == KPATH_GEMM) {   // large tiles: host walk, cuBLAS products (scratch behind the table area of the workspace)
    std::vector<WorkItem> its((size_t)n_tiles);
    for (int64_t i = 0; i < n_tiles; ++i) its[(size_t)i] = WorkItem{0, (int)i, 0, 0};
    long long   n_launch = 0;
    cudaError_t eg = cudaMemcpyAsync(ws, &D, sizeof(D), cudaMemcpyHostToDevice, s);
    if (eg != cudaSuccess) return cuda_fail(eg, "ns_tiles: layer table");
    // one tile per sub-batch: an implicit work list is not available on the device, so each tile is one whole block
    eg = run_gemm_path(&D, its.data(), (const LayerDev*)ws, nullptr, n_tiles, T, T, MODE_PHI, dtype, hp,
                       ws + align_up(128 + 3 * sizeof(CUtensorMap), 256), gemm_path_scratch_bytes(512, 512), s, &n_launch);
    g_launches.fetch_add(n_launch);
    if (eg != cudaSuccess) return cuda_fail(eg, "ns_tiles: large-tile path (cuBLAS)");
    return HIMUON_OK;
  }
  cudaError_t e = cudaMemcpyAsync(ws, &D, sizeof(D), cudaMemcpyHostToDevice, s);
  if (e != cudaSuccess) return cuda_fail(e, "ns_tiles: layer table");
  if (kpath_uses_tma(kp)) {
    CUtensorMap maps[3];
    std::memset(maps, 0, sizeof(maps));
    if (!encode_bf16_map(&maps[0], D.w, D.H, D.W, T, T > 128 ? 128 : T) || !encode_bf16_map(&maps[1], D.g, D.H, D.W, T, T > 128 ? 128 : T)) {
      g_last_cuda_error = "ns_tiles: cuTensorMapEncodeTiled failed or unavailable";
      return HIMUON_ERR_CUDA;
    }
    e = cudaMemcpyAsync(ws + 128, maps, sizeof(maps), cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return cuda_fail(e, "ns_tiles: tensor maps");
  }
  LaunchArgs la;
  la.layers = (const LayerDev*)ws;
  la.tmaps = (const CUtensorMap*)(ws + 128);
  la.items = nullptr;
  la.n_items = n_tiles;
  la.T = T;
  la.mode = MODE_PHI;
  la.dtype = dtype;
  la.hp = hp;
  e = launch_chunk(la, kp, s);
  if (e != cudaSuccess) return cuda_fail(e, "ns_tiles: kernel launch");
  return HIMUON_OK;
}

}  // extern "C"

// ---- himuon_ns_tiles_static: the packed-tiles entry point for callers that cannot allocate --------------------------
// Same computation as himuon_ns_tiles on bf16 storage / HIMUON_PATH_AUTO, but the device scratch
// (layer table, tensor maps, the large-tile path's operand arrays) is this file-scope array instead of a caller
// workspace: no cudaMalloc / cudaFree / allocating library call on this path, ever.  Every GPU that loads the library
// holds HIMUON_STATIC_SCRATCH_BYTES of device memory until the process exits.
namespace {

static __device__ __align__(256) unsigned char g_static_scratch[HIMUON_STATIC_SCRATCH_BYTES];

constexpr size_t kStaticTableBytes = 1024;     // layer table (128 B) + 3 tensor maps, rounded up

// Device address of g_static_scratch on the CURRENT device.  In host code the array's name is only a handle for
// cudaGetSymbolAddress, never a device pointer; the address differs per device, so it is looked up once per device
// ordinal with that device current (the caller's), under a mutex.
cudaError_t static_scratch_ptr(char** out) {
  static std::mutex mu;
  static char*      ptr[64] = {nullptr};
  int               dev = 0;
  cudaError_t       e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lock(mu);
  if (dev >= 0 && dev < 64 && ptr[dev]) { *out = ptr[dev]; return cudaSuccess; }
  void* p = nullptr;
  e = cudaGetSymbolAddress(&p, g_static_scratch);
  if (e != cudaSuccess) return e;
  if (!p) return cudaErrorInvalidSymbol;
  if (dev >= 0 && dev < 64) ptr[dev] = (char*)p;
  *out = (char*)p;
  return cudaSuccess;
}

// Scratch bytes the tiles of one call need behind the table area: only the large-tile path (T = 512) has any.
size_t static_item_bytes(int T) { return select_kpath(HIMUON_BF16, HIMUON_PATH_AUTO, T) == KPATH_LT ? lt_path_batch_item_bytes(T, T) : 0; }

}  // namespace

extern "C" {

int64_t himuon_ns_tiles_static_max_tiles(int32_t T) {
  bool known = false;
  for (int t : kTileSizes) known |= (t == T);
  if (!known || select_kpath(HIMUON_BF16, HIMUON_PATH_AUTO, T) < 0) return 0;
  const size_t  per = static_item_bytes(T);
  const int64_t by_index = 0x7fffffffLL / T;                  // tile index x T is a 32-bit row coordinate
  if (per == 0) return by_index;
  const int64_t by_scratch = (int64_t)((HIMUON_STATIC_SCRATCH_BYTES - kStaticTableBytes) / per);
  return by_scratch < by_index ? by_scratch : by_index;
}

himuon_status himuon_ns_tiles_static(const void* tiles_in, void* tiles_out, int64_t n_tiles, int32_t T, int32_t K,
                                     float a, float b, float c, float eps, void* cuda_stream) {
  if (n_tiles < 0) return HIMUON_ERR_INVALID_ARG;
  bool known = false;
  for (int t : kTileSizes) known |= (t == T);
  if (!known) return HIMUON_ERR_INVALID_ARG;
  himuon_hparams hp;
  std::memset(&hp, 0, sizeof(hp));
  hp.K = K; hp.a = a; hp.b = b; hp.c = c; hp.eps = eps;
  if (!valid_hparams(&hp)) return HIMUON_ERR_INVALID_ARG;
  const int kp = select_kpath(HIMUON_BF16, HIMUON_PATH_AUTO, T);
  if (kp < 0 || kp == KPATH_GEMM) return HIMUON_ERR_UNSUPPORTED;      // (the cuBLAS path creates a handle: it allocates)
  if (kpath_needs_positive_c(kp) && !positive_c_ok(&hp)) return HIMUON_ERR_UNSUPPORTED;
  if (n_tiles == 0) return HIMUON_OK;
  if (!tiles_in || !tiles_out) return HIMUON_ERR_INVALID_ARG;
  const int64_t max_tiles = himuon_ns_tiles_static_max_tiles(T);
  if (n_tiles > max_tiles) {
    g_last_cuda_error = "ns_tiles_static: " + std::to_string(n_tiles) + " tiles of " + std::to_string(T) + " x " + std::to_string(T) +
                        " exceed the static scratch (HIMUON_STATIC_SCRATCH_BYTES = " + std::to_string((size_t)HIMUON_STATIC_SCRATCH_BYTES) +
                        "): at most " + std::to_string(max_tiles) + " such tiles per call; split the batch or use himuon_ns_tiles";
    return HIMUON_ERR_WORKSPACE_TOO_SMALL;
  }
  if (kpath_uses_tma(kp) && (((uintptr_t)tiles_in & 15) || ((uintptr_t)tiles_out & 15))) return HIMUON_ERR_UNSUPPORTED;
  if (((uintptr_t)tiles_in & 1) || ((uintptr_t)tiles_out & 1)) return HIMUON_ERR_INVALID_ARG;

  char*       ws = nullptr;
  cudaError_t e = static_scratch_ptr(&ws);
  if (e != cudaSuccess) return cuda_fail(e, "ns_tiles_static: cudaGetSymbolAddress(static scratch)");

  // The packed batch is one (n_tiles*T) x T matrix whose tile (r, 0) is tile r.
  cudaStream_t s = (cudaStream_t)cuda_stream;
  LayerDev     D;
  D.w = tiles_out; D.g = const_cast<void*>(tiles_in); D.m = nullptr;
  D.ld_w = T; D.ld_g = T; D.ld_m = 0;
  D.H = (int)(n_tiles * T); D.W = T; D.tau_base = 0.f; D.dtype = HIMUON_BF16;
  e = cudaMemcpyAsync(ws, &D, sizeof(D), cudaMemcpyHostToDevice, s);
  if (e != cudaSuccess) return cuda_fail(e, "ns_tiles_static: layer table");
  if (kp == KPATH_LT) {     // tcgen05 GEMM path over the implicit list of the packed batch, ONE sub-batch
    long long n_launch = 0;
    e = run_lt_path(&D, nullptr, (const LayerDev*)ws, nullptr, n_tiles, T, T, MODE_PHI, hp, ws + kStaticTableBytes,
                    HIMUON_STATIC_SCRATCH_BYTES - kStaticTableBytes, s, &n_launch);
    g_launches.fetch_add(n_launch);
    if (e != cudaSuccess) return cuda_fail(e, "ns_tiles_static: large-tile path");
    return HIMUON_OK;
  }
  if (kpath_uses_tma(kp)) {
    CUtensorMap maps[3];
    std::memset(maps, 0, sizeof(maps));
    if (!encode_bf16_map(&maps[0], D.w, D.H, D.W, T, T > 128 ? 128 : T) || !encode_bf16_map(&maps[1], D.g, D.H, D.W, T, T > 128 ? 128 : T)) {
      g_last_cuda_error = "ns_tiles_static: cuTensorMapEncodeTiled failed or unavailable";
      return HIMUON_ERR_CUDA;
    }
    e = cudaMemcpyAsync(ws + 128, maps, sizeof(maps), cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return cuda_fail(e, "ns_tiles_static: tensor maps");
  }
  LaunchArgs la;
  la.layers = (const LayerDev*)ws;
  la.tmaps = (const CUtensorMap*)(ws + 128);
  la.items = nullptr;
  la.n_items = n_tiles;
  la.T = T;
  la.mode = MODE_PHI;
  la.dtype = HIMUON_BF16;
  la.hp = hp;
  e = launch_chunk(la, kp, s);
  if (e != cudaSuccess) return cuda_fail(e, "ns_tiles_static: kernel launch");
  return HIMUON_OK;
}

}  // extern "C"
