// Large-tile path of the HiMuon hot path on bf16 storage: tiles that do not fit one SM pair's on-chip memory, i.e.
// T = 512 (the paper's default tile size on A40), the full-matrix branch T >= max(H, W) beyond 256
// (the paper's T = infinity warm start), rectangular tiles (T_h, T_w) of the tile-shape
// study and T = 256 on widths TMA cannot store.  This is the paper's "multi-kernel path
// with epilogue fusion" (section 4.4.1) re-designed for sm_100a: every product of a Newton-Schulz step
// (Eq. 2.2) is ONE launch of a hand-written persistent tcgen05 GEMM over all tiles of a sub-batch,
// with the step's elementwise work fused into its epilogue - nothing but bf16 arrays (operands, the iterate as a hi + lo pair) and three
// small fp32 vectors per tile ever touches HBM between the products:
//
//   lt_prep    M' = beta M + G (stored); Ghat = G + beta M' | M' -> the iterate, kept as TWO bf16 arrays
//              Xb = bf16(Ghat) (hi: the products' operand) and Xlo = bf16(Ghat - hi) (scratch, tile zero-padded, stored
//              TRANSPOSED when the tile is tall so that the Gram matrix is on the short side); row-norm
//              partials d_i and per-block partial sums of squares (fixed summation order).  hi + lo carries 16 mantissa
//              bits (2^-17 relative, far below the operands' bf16 rounding) and costs half the HBM traffic of an fp32
//              copy beside the bf16 operand: the path is bound by HBM, every product round-trips through it.
//              The normalisation X0 = q Ghat / (||Ghat||_F + eps), q = c^(1/4) (Phi_K(0) = 0) is NOT a
//              pass of its own: bf16 rounding is scale-free, so the first step runs on the raw Ghat and its epilogues
//              apply sigma = q / (||Ghat||_F + eps) (E1: sigma^2 on the accumulator and on d; E3: sigma on the result).
//   K x  lt_gemm<E1>  ACC = Xb Xb^T;  epilogue: Ot = bf16(offdiag(ACC) + diag(d + beta/2)) -> Ob;  S_i = sum_j ACC_ij^2
//        lt_gemm<E2>  ACC = Ot Ot^T (= B off the diagonal);  epilogue: Bb = bf16(ACC), diagonal zeroed -> Bb
//        lt_gemm<E3>  ACC = Bb Xb;  epilogue: x <- sigma ((a + beta d_i + S_i) (hi + lo) + ACC) in fp32; new hi -> the
//                     other Xb, new lo in place; new d_i partials
//   lt_update  W <- (1 - lr wd) W - lr tau (hi + lo) / q (Eq. 4.6; Phi mode: W <- (hi + lo) / q),
//              un-transposed
// The numerical scheme is the one of the fused kernels (scaled state, fp32 diagonals of A and B as row scalings, the
// operand-diagonal trick), so the accuracy is the same <= 3e-2 class.
//
// lt_gemm: C[b] (M x N, fp32 in TMEM) = A[b] (M x K, K-major) * B[b]; B is K-major (N x K: Gram form) or MN-major
// (K x N: plain product).  CTA tile 128 x 256 (or 256 x 256 over a CTA pair, below), k-block 64, shared-memory stages
// filled by TMA (3-D tensor maps over the batched scratch arrays; out-of-bounds rows / columns read as zero), SS-mode
// tcgen05.mma 128 x 256 x 16 issued by one thread, two 256-column accumulators in TMEM so that the epilogue of one tile
// overlaps the products of the next; persistent over batch x tiles.  Warps: 0 = TMA producer of the operands, 1 = MMA
// issuer, 2 = TMA producer of the iterate's chunks (E3), 4-11 = epilogue: thread = accumulator row x column half, and
// every byte of the epilogue's global traffic goes through TMA (iterate chunks in, updated in place in shared memory,
// out; bf16 operands out) - tcgen05.ld hands a thread one ROW, so direct global accesses would be 32 rows per warp
// instruction.
#include <cuda_bf16.h>

#include <algorithm>
#include <cstring>

#include "himuon_internal.h"
#include "sm100_ptx.cuh"
#include "tc_common.cuh"

namespace himuon {
namespace {

using namespace ptx;
using namespace tc;

constexpr int BM = 128, BN = 256, BK = 64;
constexpr uint32_t kABytes = BM * BK * 2;
constexpr int kGemmThreads = 384;          // warps 0 / 1 / 2: operand producer / MMA issuer / iterate producer, 4-11 epilogue
constexpr int kEpiThreads = 256;
constexpr int kEwThreads = 256;
constexpr int kPrepBlocks = 32;          // blocks per tile of lt_prep / lt_update (fixed: summation order)

inline long long rup(long long x, long long a) { return (x + a - 1) / a * a; }

// Geometry of one sub-batch: nb tiles of Th x Tw (storage orientation), iterated as rp x np with rp <= np.
struct LtGeom {
  int Th, Tw;            // tile extent in the parameter's storage (rows, columns)
  int rp, np;            // iterate extent: (Th, Tw) or, transposed, (Tw, Th); multiples of 8
  int transposed;        // 1: the iterate is the transposed tile
  int ldx, ldr;          // leading dimensions of the [rp x np] and [rp x rp] scratch arrays (elements)
  int ntx, ntr;          // BN-column slots of an [.. x np] / [.. x rp] array (partial-sum slots)
  long long sx, sr;      // per-tile strides of the [rp x ldx] / [rp x ldr] arrays (elements)
  long long sd, ss;      // per-tile strides of the d / S partial arrays (floats)
};

LtGeom make_geom(int Th, int Tw) {
  LtGeom g;
  g.Th = Th; g.Tw = Tw;
  g.transposed = Th > Tw;
  g.rp = (int)rup(std::min(Th, Tw), 8);
  g.np = (int)rup(std::max(Th, Tw), 8);
  g.ldx = (int)rup(g.np, 64);
  g.ldr = (int)rup(g.rp, 64);
  g.ntx = (g.np + BN - 1) / BN;            // partial-sum slots: one per BN-column tile of the output
  g.ntr = (g.rp + BN - 1) / BN;
  g.sx = (long long)g.rp * g.ldx;
  g.sr = (long long)g.rp * g.ldr;
  g.sd = (long long)g.ntx * g.rp;
  g.ss = (long long)g.ntr * g.rp;
  return g;
}

size_t a256(size_t x) { return (x + 255) & ~(size_t)255; }

// Scratch of a sub-batch of nb tiles: Xb x 2, Xlo, Ob, Bb (bf16), d partials x 2 (ping-pong), S partials, ss partials.
struct LtScratch {
  __nv_bfloat16 *xlo, *xb, *xb2, *ob, *bb; float *d0, *d1, *sp, *ssq;   // xb / xb2: product 3 reads one, writes the other
};
size_t lt_item_bytes(const LtGeom& g) {
  return 3 * a256((size_t)g.sx * 2) + 2 * a256((size_t)g.sr * 2) + 2 * a256((size_t)g.sd * 4) +
         a256((size_t)g.ss * 4) + a256(kPrepBlocks * 4);
}
LtScratch carve(char* base, const LtGeom& g, int nb) {
  LtScratch s;
  size_t off = 0;
  auto take = [&](size_t per) { char* p = base + off; off += (size_t)nb * per; return p; };
  s.xlo = (__nv_bfloat16*)take(a256((size_t)g.sx * 2));
  s.xb = (__nv_bfloat16*)take(a256((size_t)g.sx * 2));
  s.xb2 = (__nv_bfloat16*)take(a256((size_t)g.sx * 2));
  s.ob = (__nv_bfloat16*)take(a256((size_t)g.sr * 2));
  s.bb = (__nv_bfloat16*)take(a256((size_t)g.sr * 2));
  s.d0 = (float*)take(a256((size_t)g.sd * 4));
  s.d1 = (float*)take(a256((size_t)g.sd * 4));
  s.sp = (float*)take(a256((size_t)g.ss * 4));
  s.ssq = (float*)take(a256(kPrepBlocks * 4));
  return s;
}
// per-tile strides in ELEMENTS of the carved arrays (the a256 rounding is per tile)
long long stride_xb(const LtGeom& g) { return (long long)(a256((size_t)g.sx * 2) / 2); }
long long stride_r(const LtGeom& g) { return (long long)(a256((size_t)g.sr * 2) / 2); }
long long stride_d(const LtGeom& g) { return (long long)(a256((size_t)g.sd * 4) / 4); }
long long stride_s(const LtGeom& g) { return (long long)(a256((size_t)g.ss * 4) / 4); }

// ---- the tile of a work item -----------------------------------------------------------------------------------
struct TileRef {
  const __nv_bfloat16* g;
  __nv_bfloat16* m;
  __nv_bfloat16* w;
  long long ld_g, ld_m, ld_w;
  int h, w_;             // live extent (rows, columns) of this tile in the parameter
  float tau_base;
};
__device__ __forceinline__ TileRef tile_ref(const LayerDev* layers, const WorkItem* items, int b, int Th, int Tw, int whole) {
  // items == nullptr: implicit list of a packed [N, T, T] batch (himuon_ns_tiles): item i = (layer 0, r = i, c = 0);
  // `whole` then carries the index of the sub-batch's first tile (and is never the whole-matrix flag)
  const WorkItem wi = items ? items[b] : WorkItem{0, whole + b, 0, 0};
  if (!items) whole = 0;
  const LayerDev L = layers[wi.layer];
  TileRef t;
  const long long row0 = whole ? 0 : (long long)wi.r * Th, col0 = whole ? 0 : (long long)wi.c * Tw;
  t.h = (int)min((long long)Th, (long long)L.H - row0);
  t.w_ = (int)min((long long)Tw, (long long)L.W - col0);
  t.g = reinterpret_cast<const __nv_bfloat16*>(L.g) + row0 * L.ld_g + col0;
  t.m = L.m ? reinterpret_cast<__nv_bfloat16*>(L.m) + row0 * L.ld_m + col0 : nullptr;
  t.w = reinterpret_cast<__nv_bfloat16*>(L.w) + row0 * L.ld_w + col0;
  t.ld_g = L.ld_g; t.ld_m = L.ld_m; t.ld_w = L.ld_w;
  t.tau_base = L.tau_base;
  return t;
}

// ---- fused ends ------------------------------------------------------------------------------------------------
// sigma = q / (||Ghat||_F + eps) of tile b from the tile's sum of squares (slot 0 of its ssq entry: lt_ssq_fold /
// lt_ssq_from_d put it there in one fixed summation order).
__device__ __forceinline__ float sigma_of(float tot, float eps, float qs) {
  const float nrm = sqrtf(tot);
  return nrm > 0.f ? qs / (nrm + eps) : 0.f;          // Phi_K(0) = 0
}
__device__ __forceinline__ float tile_sigma(const float* __restrict__ ssq, int b, float eps, float qs) {
  return sigma_of(ssq[(long long)b * kPrepBlocks], eps, qs);
}
// lt_prep's per-block partial sums of a tile, added in block order, into slot 0 (one thread per tile: the GEMM
// epilogues and lt_update then need one load per tile, not kPrepBlocks of them per thread and work unit)
__global__ void lt_ssq_fold(float* __restrict__ ssq, int nb) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= nb) return;
  float tot = 0.f;
#pragma unroll
  for (int i = 0; i < kPrepBlocks; ++i) tot += ssq[(long long)b * kPrepBlocks + i];
  ssq[(long long)b * kPrepBlocks] = tot;
}

// 16-byte accesses of a tile: base pointers, leading dimensions and live width all multiples of 8 bf16
__device__ __forceinline__ bool tile_vec8(const TileRef& t, bool with_m) {
  bool ok = (t.w_ % 8 == 0) && (t.ld_g % 8 == 0) && (t.ld_w % 8 == 0) && ((reinterpret_cast<uintptr_t>(t.g) & 15) == 0) &&
            ((reinterpret_cast<uintptr_t>(t.w) & 15) == 0);
  if (with_m) ok = ok && (t.ld_m % 8 == 0) && ((reinterpret_cast<uintptr_t>(t.m) & 15) == 0);
  return ok;
}
__device__ __forceinline__ void unpack8(const uint4 v, float (&f)[8]) {
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    f[2 * k] = __uint_as_float(w[k] << 16);
    f[2 * k + 1] = __uint_as_float(w[k] & 0xffff0000u);
  }
}
__device__ __forceinline__ uint4 pack8(const float (&f)[8]) {
  return make_uint4(pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
}

// grid (kPrepBlocks, nb) (big tiles: more blocks, ssq == nullptr), one warp per row of the SCRATCH layout (rp x ldx, coalesced writes); element (i, j) of the
// iterate is element (i, j) of the tile, or (j, i) when transposed.  Untransposed tiles whose rows are 16-byte aligned
// take the wide path: a lane owns 8 consecutive columns of a BN-column slot, both loads of a slot pair are issued
// before the first store (the stores to M could alias the loads of G for all the compiler knows).
__global__ void __launch_bounds__(kEwThreads)
lt_prep(const LayerDev* __restrict__ layers, const WorkItem* __restrict__ items, LtGeom g, int whole,
        __nv_bfloat16* __restrict__ xlo, __nv_bfloat16* __restrict__ xb, long long sxb, float* __restrict__ d0, long long sd,
        float* __restrict__ ssq, int step_mode, float beta, int nesterov) {
  const int b = blockIdx.y;
  const TileRef t = tile_ref(layers, items, b, g.Th, g.Tw, whole);
  __nv_bfloat16* Xl = xlo + (long long)b * sxb;
  __nv_bfloat16* Xb = xb + (long long)b * sxb;
  float* D = d0 + (long long)b * sd;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  float ss = 0.f;
  if (!g.transposed && tile_vec8(t, step_mode != 0)) {
    for (int i = blockIdx.x * (kEwThreads / 32) + warp; i < g.rp; i += (int)gridDim.x * (kEwThreads / 32)) {
      const bool row_ok = i < t.h;
      for (int slot0 = 0; slot0 < g.ntx; slot0 += 2) {
        uint4 gv[2], mv[2];
        bool live[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          const int j = (slot0 + u) * BN + 8 * lane;
          live[u] = row_ok && slot0 + u < g.ntx && j < t.w_;
          gv[u] = make_uint4(0, 0, 0, 0);
          mv[u] = make_uint4(0, 0, 0, 0);
          if (live[u]) {
            gv[u] = *reinterpret_cast<const uint4*>(t.g + (long long)i * t.ld_g + j);
            if (step_mode) mv[u] = *reinterpret_cast<const uint4*>(t.m + (long long)i * t.ld_m + j);
          }
        }
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          const int slot = slot0 + u, j = slot * BN + 8 * lane;
          if (slot >= g.ntx) break;
          float x[8];
          unpack8(gv[u], x);                                                 // outside the tile: zeros (B_T padding)
          if (step_mode && live[u]) {
            float m[8];
            unpack8(mv[u], m);
#pragma unroll
            for (int k = 0; k < 8; ++k) m[k] = fmaf(beta, m[k], x[k]);
            *reinterpret_cast<uint4*>(t.m + (long long)i * t.ld_m + j) = pack8(m);
#pragma unroll
            for (int k = 0; k < 8; ++k) x[k] = nesterov ? fmaf(beta, m[k], x[k]) : m[k];
          }
          float dd = 0.f;
          if (j < g.ldx) {
            const uint4 hi = pack8(x);
            float h[8], l[8];
            unpack8(hi, h);
#pragma unroll
            for (int k = 0; k < 8; ++k) l[k] = x[k] - h[k];
            *reinterpret_cast<uint4*>(Xb + (long long)i * g.ldx + j) = hi;
            *reinterpret_cast<uint4*>(Xl + (long long)i * g.ldx + j) = pack8(l);
#pragma unroll
            for (int k = 0; k < 8; ++k) dd = fmaf(x[k], x[k], dd);
          }
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) dd += __shfl_xor_sync(0xffffffffu, dd, o);
          if (lane == 0) D[(long long)slot * g.rp + i] = dd;
          ss += dd;                                      // identical in every lane
        }
      }
    }
  } else {
    for (int i = blockIdx.x * (kEwThreads / 32) + warp; i < g.rp; i += (int)gridDim.x * (kEwThreads / 32)) {
      for (int slot = 0; slot < g.ntx; ++slot) {        // d partial per BN-column slot, as the E3 epilogue writes them
        float dd = 0.f;
        const int j1 = min((slot + 1) * BN, g.ldx);
        for (int j = slot * BN + lane; j < j1; j += 32) {
          const int r = g.transposed ? j : i, c = g.transposed ? i : j;    // position in the tile
          float x = 0.f;
          if (r < t.h && c < t.w_) {                                         // outside: B_T zero padding
            const float gg = __bfloat162float(t.g[(long long)r * t.ld_g + c]);
            x = gg;
            if (step_mode) {
              __nv_bfloat16* pm = t.m + (long long)r * t.ld_m + c;
              const float mm = fmaf(beta, __bfloat162float(*pm), gg);
              *pm = __float2bfloat16_rn(mm);
              x = nesterov ? fmaf(beta, mm, gg) : mm;
            }
          }
          const __nv_bfloat16 hi = __float2bfloat16_rn(x);
          Xb[(long long)i * g.ldx + j] = hi;
          Xl[(long long)i * g.ldx + j] = __float2bfloat16_rn(x - __bfloat162float(hi));
          dd = fmaf(x, x, dd);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) dd += __shfl_xor_sync(0xffffffffu, dd, o);
        if (lane == 0) D[(long long)slot * g.rp + i] = dd;
        ss += dd;                                        // identical in every lane
      }
    }
  }
  __shared__ float red[kEwThreads / 32];
  if (lane == 0) red[warp] = ss;
  __syncthreads();
  if (threadIdx.x == 0 && ssq) {      // (big tiles run on a wider grid and take the sum from the d partials: lt_ssq_from_d)
    float tot = 0.f;
#pragma unroll
    for (int i = 0; i < kEwThreads / 32; ++i) tot += red[i];
    ssq[(long long)b * kPrepBlocks + blockIdx.x] = tot;
  }
}

__global__ void __launch_bounds__(kEwThreads)
lt_update(const LayerDev* __restrict__ layers, const WorkItem* __restrict__ items, LtGeom g, int whole,
          const __nv_bfloat16* __restrict__ xhi, const __nv_bfloat16* __restrict__ xlo, long long sxb, int step_mode, float keep,
          float lr_scale, float unq,
          const float* __restrict__ ssq, float eps, float qs) {
  const int b = blockIdx.y;
  const TileRef t = tile_ref(layers, items, b, g.Th, g.Tw, whole);
  const __nv_bfloat16* Xh = xhi + (long long)b * sxb;
  const __nv_bfloat16* Xl = xlo + (long long)b * sxb;
  const float sig = ssq ? tile_sigma(ssq, b, eps, qs) : 1.f;      // K = 0: the iterate is still the raw Ghat
  const float stepsz = (step_mode ? lr_scale * t.tau_base * unq : unq) * sig;
  if (!g.transposed && tile_vec8(t, false)) {
    // wide path: a thread owns 8 consecutive columns of a row; two such pieces in flight per thread
    const int w8 = t.w_ / 8;
    const long long n8 = (long long)t.h * w8, stride = (long long)gridDim.x * kEwThreads;
    for (long long e0 = (long long)blockIdx.x * kEwThreads + threadIdx.x; e0 < n8; e0 += 2 * stride) {
      uint4 xh[2], xl[2];
      uint4 wv[2];
      __nv_bfloat16* pw[2];
      bool live[2];
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const long long e = e0 + u * stride;
        live[u] = e < n8;
        if (live[u]) {
          const int r = (int)(e / w8), c = 8 * (int)(e - (long long)r * w8);
          xh[u] = __ldcs(reinterpret_cast<const uint4*>(Xh + (long long)r * g.ldx + c));
          xl[u] = __ldcs(reinterpret_cast<const uint4*>(Xl + (long long)r * g.ldx + c));
          pw[u] = t.w + (long long)r * t.ld_w + c;
          if (step_mode) wv[u] = *reinterpret_cast<const uint4*>(pw[u]);
        }
      }
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        if (!live[u]) continue;
        float x[8], xq[8];
        unpack8(xh[u], x);
        unpack8(xl[u], xq);
#pragma unroll
        for (int k = 0; k < 8; ++k) x[k] += xq[k];
        float o[8];
        if (step_mode) {
          unpack8(wv[u], o);
#pragma unroll
          for (int k = 0; k < 8; ++k) o[k] = fmaf(keep, o[k], stepsz * x[k]);
        } else {
#pragma unroll
          for (int k = 0; k < 8; ++k) o[k] = stepsz * x[k];
        }
        *reinterpret_cast<uint4*>(pw[u]) = pack8(o);
      }
    }
    return;
  }
  const long long n = (long long)t.h * t.w_;
  for (long long e = (long long)blockIdx.x * kEwThreads + threadIdx.x; e < n; e += (long long)gridDim.x * kEwThreads) {
    const int r = (int)(e / t.w_), c = (int)(e - (long long)r * t.w_);
    const long long at = g.transposed ? (long long)c * g.ldx + r : (long long)r * g.ldx + c;
    const float x = __bfloat162float(Xh[at]) + __bfloat162float(Xl[at]);
    __nv_bfloat16* p = t.w + (long long)r * t.ld_w + c;
    *p = __float2bfloat16_rn(step_mode ? fmaf(keep, __bfloat162float(*p), stepsz * x) : stepsz * x);
  }
}

// ---- fused ends of BIG tiles (the full-matrix branch, tiles of >= 1 M elements) ----------------------------------------
// With one tile (or a few) per sub-batch the kPrepBlocks x nb grid of lt_prep / lt_update is a fraction of the GPU, and the
// scalar path of a TRANSPOSED tile touches one 2-byte element per lane and row (measured on a 14336 x 4096 matrix: 6.3 ms
// of lt_prep + 4.3 ms of lt_update beside 4.2 ms for the fifteen GEMMs).  Big tiles therefore run lt_prep / lt_update on a
// grid sized by the tile, transposed tiles (of any size) go through the two kernels below (64 x 64 patches transposed in shared
// memory: every global access is a row segment in BOTH layouts), and the sum of squares of the tile comes from the d
// partials in one fixed order (lt_ssq_from_d).
constexpr int kTP = 64;                   // patch edge

// 16 consecutive bf16 -> fp32 (the first nv of them; the rest read as zero) and back; 16-byte accesses when `vec`
__device__ __forceinline__ void load16(const __nv_bfloat16* p, int nv, bool vec, float (&f)[16]) {
  if (vec && nv == 16) {
    float a[8], b[8];
    unpack8(*reinterpret_cast<const uint4*>(p), a);
    unpack8(*reinterpret_cast<const uint4*>(p + 8), b);
#pragma unroll
    for (int k = 0; k < 8; ++k) { f[k] = a[k]; f[8 + k] = b[k]; }
  } else {
#pragma unroll
    for (int k = 0; k < 16; ++k) f[k] = k < nv ? __bfloat162float(p[k]) : 0.f;
  }
}
__device__ __forceinline__ void store16(__nv_bfloat16* p, int nv, bool vec, const float (&f)[16]) {
  if (vec && nv == 16) {
    const float a[8] = {f[0], f[1], f[2], f[3], f[4], f[5], f[6], f[7]};
    const float b[8] = {f[8], f[9], f[10], f[11], f[12], f[13], f[14], f[15]};
    *reinterpret_cast<uint4*>(p) = pack8(a);
    *reinterpret_cast<uint4*>(p + 8) = pack8(b);
  } else {
#pragma unroll
    for (int k = 0; k < 16; ++k)
      if (k < nv) p[k] = __float2bfloat16_rn(f[k]);
  }
}

// lt_prep for transposed tiles: iterate (i, j) = tile (j, i).  grid (ceil(rp / 64), ntx, nb), 256 threads; a block owns
// iterate rows C0 .. C0 + 63 (tile columns) and the iterate columns of d-partial slot blockIdx.y (tile rows), 64 at a time.
__global__ void __launch_bounds__(kEwThreads)
lt_prep_t(const LayerDev* __restrict__ layers, const WorkItem* __restrict__ items, LtGeom g, int whole,
          __nv_bfloat16* __restrict__ xlo, __nv_bfloat16* __restrict__ xb, long long sxb, float* __restrict__ d0, long long sd,
          int step_mode, float beta, int nesterov) {
  const int b = blockIdx.z;
  const TileRef t = tile_ref(layers, items, b, g.Th, g.Tw, whole);
  __nv_bfloat16* Xl = xlo + (long long)b * sxb;
  __nv_bfloat16* Xb = xb + (long long)b * sxb;
  float* D = d0 + (long long)b * sd;
  const int slot = blockIdx.y, C0 = blockIdx.x * kTP;
  const int rr = threadIdx.x >> 2, seg = threadIdx.x & 3;
  const bool vec = tile_vec8(t, step_mode != 0);
  __shared__ float xs[kTP][kTP + 1];
  float dd = 0.f;                          // this thread's share of sum_j x_ij^2, i = C0 + rr, j in the slot
  const int jend = min((slot + 1) * BN, g.ldx);
  for (int R0 = slot * BN; R0 < jend; R0 += kTP) {
    {   // tile row R0 + rr, tile columns C0 + 16 seg .. + 15: momentum in the tile's own layout
      const int r = R0 + rr, c0 = C0 + 16 * seg;
      float x[16];
#pragma unroll
      for (int k = 0; k < 16; ++k) x[k] = 0.f;                               // outside the tile: B_T zero padding
      if (r < t.h && c0 < t.w_) {
        const int nv = min(16, t.w_ - c0);
        load16(t.g + (long long)r * t.ld_g + c0, nv, vec, x);
        if (step_mode) {
          float m[16];
          __nv_bfloat16* pm = t.m + (long long)r * t.ld_m + c0;
          load16(pm, nv, vec, m);
#pragma unroll
          for (int k = 0; k < 16; ++k) m[k] = fmaf(beta, m[k], x[k]);
          store16(pm, nv, vec, m);
#pragma unroll
          for (int k = 0; k < 16; ++k) x[k] = k < nv ? (nesterov ? fmaf(beta, m[k], x[k]) : m[k]) : 0.f;
        }
      }
#pragma unroll
      for (int k = 0; k < 16; ++k) xs[16 * seg + k][rr] = x[k];
    }
    __syncthreads();
    {   // iterate row C0 + rr, iterate columns R0 + 16 seg .. + 15 (ldx is a multiple of 64: whole segments)
      const int i = C0 + rr, j0 = R0 + 16 * seg;
      if (i < g.rp) {
        float h[16], l[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) {
          const float x = xs[rr][16 * seg + k];
          h[k] = __bfloat162float(__float2bfloat16_rn(x));
          l[k] = x - h[k];
          dd = fmaf(x, x, dd);
        }
        store16(Xb + (long long)i * g.ldx + j0, 16, true, h);
        store16(Xl + (long long)i * g.ldx + j0, 16, true, l);
      }
    }
    __syncthreads();
  }
  dd += __shfl_xor_sync(0xffffffffu, dd, 1);
  dd += __shfl_xor_sync(0xffffffffu, dd, 2);
  if (seg == 0 && C0 + rr < g.rp) D[(long long)slot * g.rp + C0 + rr] = dd;
}

// lt_update for transposed tiles.  grid (ceil(rp / 64), ceil(np / 64), nb), 256 threads.
__global__ void __launch_bounds__(kEwThreads)
lt_update_t(const LayerDev* __restrict__ layers, const WorkItem* __restrict__ items, LtGeom g, int whole,
            const __nv_bfloat16* __restrict__ xhi, const __nv_bfloat16* __restrict__ xlo, long long sxb, int step_mode, float keep,
            float lr_scale, float unq, const float* __restrict__ ssq, float eps, float qs) {
  const int b = blockIdx.z;
  const TileRef t = tile_ref(layers, items, b, g.Th, g.Tw, whole);
  const __nv_bfloat16* Xh = xhi + (long long)b * sxb;
  const __nv_bfloat16* Xl = xlo + (long long)b * sxb;
  const float sig = ssq ? tile_sigma(ssq, b, eps, qs) : 1.f;      // K = 0: the iterate is still the raw Ghat
  const float stepsz = (step_mode ? lr_scale * t.tau_base * unq : unq) * sig;
  const int C0 = blockIdx.x * kTP, R0 = blockIdx.y * kTP;
  const int rr = threadIdx.x >> 2, seg = threadIdx.x & 3;
  __shared__ float xs[kTP][kTP + 1];
  {   // iterate row C0 + rr, iterate columns R0 + 16 seg .. + 15
    const int i = C0 + rr, j0 = R0 + 16 * seg;
    float h[16], l[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) h[k] = l[k] = 0.f;
    if (i < g.rp && j0 < g.ldx) {
      load16(Xh + (long long)i * g.ldx + j0, 16, true, h);
      load16(Xl + (long long)i * g.ldx + j0, 16, true, l);
    }
#pragma unroll
    for (int k = 0; k < 16; ++k) xs[rr][16 * seg + k] = h[k] + l[k];
  }
  __syncthreads();
  {   // tile row R0 + rr, tile columns C0 + 16 seg .. + 15
    const int r = R0 + rr, c0 = C0 + 16 * seg;
    if (r < t.h && c0 < t.w_) {
      const int nv = min(16, t.w_ - c0);
      const bool vec = tile_vec8(t, false);
      __nv_bfloat16* pw = t.w + (long long)r * t.ld_w + c0;
      float o[16];
      if (step_mode) {
        load16(pw, nv, vec, o);
#pragma unroll
        for (int k = 0; k < 16; ++k) o[k] = fmaf(keep, o[k], stepsz * xs[16 * seg + k][rr]);
      } else {
#pragma unroll
        for (int k = 0; k < 16; ++k) o[k] = stepsz * xs[16 * seg + k][rr];
      }
      store16(pw, nv, vec, o);
    }
  }
}

// ||Ghat||_F^2 of every tile from its d partials (row sums of squares), in one fixed order -> the slot layout tile_sigma reads
__global__ void __launch_bounds__(1024)
lt_ssq_from_d(const float* __restrict__ d0, long long sd, int n, float* __restrict__ ssq) {
  const int b = blockIdx.x;
  const float* D = d0 + (long long)b * sd;
  __shared__ float red[1024];
  float s = 0.f;
  for (int e = threadIdx.x; e < n; e += 1024) s += D[e];
  red[threadIdx.x] = s;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x < kPrepBlocks) ssq[(long long)b * kPrepBlocks + threadIdx.x] = threadIdx.x == 0 ? red[0] : 0.f;
}

// ---- the GEMM --------------------------------------------------------------------------------------------------
enum { EPI_GRAM = 1, EPI_B = 2, EPI_X = 3 };

struct GemmParams {
  int M, N, K;                 // C[b] is M x N; K = contraction length (all multiples of 8)
  int nb, mt, nt;              // batch, tiles per batch item
  const float* d_in;           // d partials of the current iterate: [b][ntx][rp]
  float* d_out;                // E3: d partials of the new iterate
  long long sd;
  int ntx;
  float* s_part;               // S partials: [b][ntr][rp]  (E1 writes, E3 reads)
  long long ss;
  int ntr;
  int rp;
  float a, beta_h;
  const float* ssq;            // first step only (else null): the iterate is still the raw Ghat, apply sigma here
  float eps, qs;
};

// Shared memory: operand stages (A: 16 KB; B: 32 KB, or 16 KB per CTA of a pair), then the epilogue staging.
//   E1 / E2: 4 stages (pair: 6) - the mainloop is bound by bytes in flight per SM (stage bytes / TMA round trip), every
//            stage counts; two alternating 16 KB buffers, one [128 rows x 64 bf16] output chunk each (128-byte swizzle,
//            the layout of the operand tiles).
//   E3:      3 stages (pair: 4); kXBufs 16 KB buffers = one [128 rows x 32 columns] chunk of the iterate each, as its two
//            bf16 halves (hi at +0, lo at +8 KB; rows of 64 B, 64-byte swizzle): TMA in, updated in place, TMA out.  E3 is
//            bound by the iterate's HBM traffic, so the rest of the shared memory goes to chunk loads in flight
//            (kXBufs - 1 chunks ahead of the epilogue).
constexpr uint32_t kEpiBuf = 16384;
constexpr int kMaxXBufs = 6;
constexpr int kMaxStages = 6;
template <int EPI, bool PAIR> struct Cfg {
  static constexpr int kStages = EPI == 3 ? (PAIR ? 4 : 3) : (PAIR ? 6 : 4);
  static constexpr int kXBufs = PAIR ? 6 : 5;
  static constexpr int kBRows = PAIR ? BN / 2 : BN;                  // rows (n) of B held by one CTA
  static constexpr uint32_t kBBytes = kBRows * BK * 2, kStageBytes = kABytes + kBBytes;
  static constexpr uint32_t kEpiBytes = EPI == 3 ? kXBufs * kEpiBuf : 2 * kEpiBuf;
  static constexpr uint32_t kSmem = kStages * kStageBytes + kEpiBytes + 1024 + 1024;
};
struct GemmCtrl {
  unsigned long long full[kMaxStages], empty[kMaxStages], tfull[2], tempty[2], xfull[kMaxXBufs], xfree[kMaxXBufs];
  uint32_t tmem_base;
  float red[BM];             // row sums of the upper column halves, handed to the lower halves' threads
};

// PAIR: two CTAs of a cluster work on one 256 x 256 tile with cta_group::2 MMAs (M = 256: 128 rows per CTA, each in its
// own TMEM; N = 256: each CTA's shared memory holds half of B), so a CTA fetches 32 KB per k-block instead of 48 KB for
// the same 128 x 256 x 64 of work - the single-CTA mainloop is bound by L2 / shared-memory fill bandwidth (96 B per
// clock and SM), not by the tensor pipe.  Every CTA runs its own TMA producer into its own stages, both counting their
// bytes on the LEADER's "stage full" barrier; the leader's MMA warp issues for both, commits are multicast to both.  The
// epilogues are per CTA (its 128 rows) and identical to the single-CTA kernel's.
template <int EPI, bool B_MN, bool PAIR>
__global__ void __launch_bounds__(kGemmThreads, 1)
lt_gemm(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const __grid_constant__ CUtensorMap tmOut,
        const __grid_constant__ CUtensorMap tmHi, const __grid_constant__ CUtensorMap tmLo, const GemmParams p) {
  using C = Cfg<EPI, PAIR>;
  constexpr int kStages = C::kStages;
  constexpr uint32_t kEpiBytes = C::kEpiBytes, kStageBytes = C::kStageBytes;
  constexpr int kXBufs = C::kXBufs;
  constexpr int kUnitM = PAIR ? 2 * BM : BM;                       // rows of C per work unit
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t epi0 = smem0 + kStages * kStageBytes;
  GemmCtrl* ctrl = reinterpret_cast<GemmCtrl*>(smem_raw + (smem0 - smem_u32(smem_raw)) + kStages * kStageBytes + kEpiBytes);
  const int tid = threadIdx.x;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int lane = tid & 31;
  const uint32_t rank = PAIR ? cluster_ctarank() : 0u;            // PAIR: 0 = leader (issues the MMAs)
  const long long unit0 = PAIR ? cluster_id_x() : blockIdx.x, unit_stride = PAIR ? cluster_count_x() : gridDim.x;

  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) {
      mbar_init(smem_u32(&ctrl->full[s]), 1);
      mbar_init(smem_u32(&ctrl->empty[s]), 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(smem_u32(&ctrl->tfull[a]), 1);
      mbar_init(smem_u32(&ctrl->tempty[a]), (PAIR ? 2 : 1) * kEpiThreads);      // PAIR: the leader's barrier collects both epilogues
    }
    for (int a = 0; a < kXBufs; ++a) {
      mbar_init(smem_u32(&ctrl->xfull[a]), 1);
      mbar_init(smem_u32(&ctrl->xfree[a]), 1);
    }
    fence_mbar_init();
  }
  if (PAIR) {
    cluster_sync_all();                                           // both CTAs' barriers exist before anyone signals
    if (warp == 1) tmem_alloc_pair<512>(smem_u32(&ctrl->tmem_base));
    tc_fence_before_sync();
    cluster_sync_all();
  } else {
    if (warp == 1) tmem_alloc<512>(smem_u32(&ctrl->tmem_base));
    tc_fence_before_sync();
    __syncthreads();
  }
  tc_fence_after_sync();
  const uint32_t tmem_base = ctrl->tmem_base;

  const long long n_tiles = (long long)p.nb * p.mt * p.nt;
  const int kb_n = (p.K + BK - 1) / BK;

  if (warp == 0) {
    // ================= TMA producer: operands =================
    if (elect_one()) {
      prefetch_tmap(&tmA);
      prefetch_tmap(&tmB);
      int s = 0;
      uint32_t ph = 0;
      for (long long tile = unit0; tile < n_tiles; tile += unit_stride) {
        const int b = (int)(tile / (p.mt * p.nt)), rem = (int)(tile - (long long)b * p.mt * p.nt);
        const int m0 = (rem / p.nt) * kUnitM + (int)rank * BM, n0 = (rem % p.nt) * BN;
        for (int kb = 0; kb < kb_n; ++kb) {
          // slot free (first pass: passes immediately).  A barrier completed by the LEADER's multicast commit does not
          // wake a parked thread of the peer before its hint expires (measured: 1 us per k-block): spin in pair mode.
          if (PAIR) mbar_wait(smem_u32(&ctrl->empty[s]), ph ^ 1);
          else mbar_wait_parked(smem_u32(&ctrl->empty[s]), ph ^ 1);
          // PAIR: both CTAs' loads count on the LEADER's barrier (armed by the leader for both stages' bytes)
          const uint32_t full = PAIR ? mapa_shared(smem_u32(&ctrl->full[s]), 0) : smem_u32(&ctrl->full[s]);
          const uint32_t sa = smem0 + s * kStageBytes, sbm = sa + kABytes;
          if (rank == 0) mbar_arrive_expect_tx(smem_u32(&ctrl->full[s]), (PAIR ? 2 : 1) * kStageBytes);
          auto load = [&](uint32_t dst, const CUtensorMap* tm, int x, int y) {
            if (PAIR) tma_load_3d_pair(dst, tm, x, y, b, full);
            else tma_load_3d(dst, tm, x, y, b, full);
          };
          load(sa, &tmA, kb * BK, m0);                                        // A: [BM rows x 64 k]
          const int nb0 = n0 + (int)rank * C::kBRows;                         // PAIR: this CTA's half of the tile's columns
          if (!B_MN) {
            load(sbm, &tmB, kb * BK, nb0);                                    // B K-major: [kBRows rows x 64 k]
          } else {
#pragma unroll
            for (int j = 0; j < C::kBRows / 64; ++j)                          // B MN-major: [64 k-rows x 64 n] boxes
              load(sbm + j * (BK * 128), &tmB, nb0 + 64 * j, kb * BK);
          }
          if (++s == kStages) { s = 0; ph ^= 1; }
        }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // ================= MMA issuer (PAIR: of the leader; the peer's warp relays its "stage full") =================
    if (PAIR && rank != 0) {
      // the peer's tensor core is driven by the leader's instructions
    } else if (elect_one()) {
      const uint32_t idesc = make_idesc_bf16(kUnitM, BN, 0, B_MN ? 1 : 0);
      int s = 0;
      uint32_t ph = 0;
      uint32_t tph[2] = {0, 0};
      int it = 0;
      for (long long tile = unit0; tile < n_tiles; tile += unit_stride, ++it) {
        const int ab = it & 1;
        // the epilogue(s) have drained this accumulator
        if (PAIR) mbar_wait(smem_u32(&ctrl->tempty[ab]), tph[ab] ^ 1);
        else mbar_wait_parked(smem_u32(&ctrl->tempty[ab]), tph[ab] ^ 1);
        tph[ab] ^= 1;
        tc_fence_after_sync();
        const uint32_t acc = tmem_base + ab * BN;
        for (int kb = 0; kb < kb_n; ++kb) {
          mbar_wait_parked(smem_u32(&ctrl->full[s]), ph);
          tc_fence_after_sync();
          const uint32_t sa = smem0 + s * kStageBytes, sbm = sa + kABytes;
#pragma unroll
          for (int kk = 0; kk < BK / 16; ++kk) {
            const uint64_t da = make_smem_desc_sw128(sa + kk * 32, 16, 1024);
            const uint64_t db = B_MN ? make_smem_desc_sw128(sbm + kk * 2048, BK * 128, 1024)
                                     : make_smem_desc_sw128(sbm + kk * 32, 16, 1024);
            if (PAIR) umma_bf16_ss_pair(acc, da, db, idesc, (kb | kk) ? 1u : 0u);
            else umma_bf16_ss(acc, da, db, idesc, (kb | kk) ? 1u : 0u);
          }
          // frees the smem slot (of both CTAs) when these MMAs have read it
          if (PAIR) umma_commit_pair(smem_u32(&ctrl->empty[s]), (uint16_t)3);
          else umma_commit(smem_u32(&ctrl->empty[s]));
          if (++s == kStages) { s = 0; ph ^= 1; }
        }
        if (PAIR) umma_commit_pair(smem_u32(&ctrl->tfull[ab]), (uint16_t)3);   // accumulator ready (in both CTAs)
        else umma_commit(smem_u32(&ctrl->tfull[ab]));
      }
    }
    __syncwarp();
  } else if (warp == 2) {
    // ================= TMA producer: chunks of the fp32 iterate for the E3 epilogue =================
    if (EPI == EPI_X && elect_one()) {
      prefetch_tmap(&tmHi);
      prefetch_tmap(&tmLo);
      uint32_t buf = 0, par = 0;                                 // chunk n lives in buffer n % kXBufs, phase (n / kXBufs) & 1
      for (long long tile = unit0; tile < n_tiles; tile += unit_stride) {
        const int b = (int)(tile / (p.mt * p.nt)), rem = (int)(tile - (long long)b * p.mt * p.nt);
        const int m0 = (rem / p.nt) * kUnitM + (int)rank * BM, n0 = (rem % p.nt) * BN;
        for (int c = 0; c < BN / 32; ++c) {
          mbar_wait_parked(smem_u32(&ctrl->xfree[buf]), par ^ 1);     // the chunk stored from this buffer has left it
          const uint32_t xfull = smem_u32(&ctrl->xfull[buf]);
          mbar_arrive_expect_tx(xfull, kEpiBuf);
          tma_load_3d(epi0 + buf * kEpiBuf, &tmHi, n0 + 32 * c, m0, b, xfull);
          tma_load_3d(epi0 + buf * kEpiBuf + kEpiBuf / 2, &tmLo, n0 + 32 * c, m0, b, xfull);
          if (++buf == kXBufs) { buf = 0; par ^= 1; }
        }
      }
    }
    __syncwarp();
  } else if (warp >= 4) {
    // ================= epilogue: 8 warps; thread = accumulator row (TMEM lane) x column half of every chunk; all
    // global traffic through TMA.  Two warps per scheduler: one warp's tcgen05.ld / shared-memory latencies hide behind
    // the other's arithmetic (with 4 warps the epilogue, not the mainloop, bounded E1 / E2: 15 % issue utilisation).
    const int wq = warp & 3;                         // TMEM lane quadrant = warp index mod 4
    const int hf = (warp - 4) >> 2;                  // column half of every chunk this thread works on
    const int row = wq * 32 + lane;                  // row of the tile
    const int et = tid - 128;                        // 0..255
    const uint32_t rsw = (uint32_t)row * 128u;       // row offset in a 128-byte-row staging buffer
    const uint32_t sw = (uint32_t)(row & 7);         // 128-byte swizzle: 16-byte chunk c lives at c ^ (row & 7)
    uint32_t tph[2] = {0, 0};
    uint32_t nchunk = 0;                             // running chunk counter
    uint32_t xbuf = 0, xpar = 0, xprev = 0;          // E3: mirrors the producer's buffer / phase; buffer of the chunk before
    int it = 0;
    // Row scalars of a work unit - the tile's sum of squares (first step), the d and S partials of this thread's row -
    // are global loads with nothing to hide behind at the top of a unit (measured: 800-5800 cycles between two units of
    // an epilogue-bound kernel).  They are therefore fetched one unit AHEAD, raw, right after the current unit's
    // accumulator has arrived, and summed at the top of the next unit (up to two partial slots each, which covers
    // T = 512; longer lists - big tiles, whose units are long anyway - are summed on the spot).
    struct Raw { float tot, d0, d1, s0, s1; };
    const bool two_slots = p.ntx <= 2 && p.ntr <= 2;
    auto fetch = [&](long long tile) {
      Raw r = {0.f, 0.f, 0.f, 0.f, 0.f};
      const int b = (int)(tile / (p.mt * p.nt)), rem = (int)(tile - (long long)b * p.mt * p.nt);
      const int mi = rem / p.nt, ni = rem % p.nt;
      const int i = mi * kUnitM + (int)rank * BM + row, n0 = ni * BN;
      const bool row_ok = i < p.M;
      if (p.ssq) r.tot = p.ssq[(long long)b * kPrepBlocks];
      if ((EPI == EPI_X && row_ok) || (EPI == EPI_GRAM && row_ok && i >= n0 && i < n0 + BN)) {
        const float* D = p.d_in + (long long)b * p.sd;
        if (two_slots) {
          r.d0 = D[i];
          if (p.ntx > 1) r.d1 = D[(long long)p.rp + i];
        } else {
          for (int sl = 0; sl < p.ntx; ++sl) r.d0 += D[(long long)sl * p.rp + i];
        }
      }
      if (EPI == EPI_X && row_ok) {
        const float* S = p.s_part + (long long)b * p.ss;
        if (two_slots) {
          r.s0 = S[i];
          if (p.ntr > 1) r.s1 = S[(long long)p.rp + i];
        } else {
          for (int sl = 0; sl < p.ntr; ++sl) r.s0 += S[(long long)sl * p.rp + i];
        }
      }
      return r;
    };
    Raw cur = {0.f, 0.f, 0.f, 0.f, 0.f};
    if (unit0 < n_tiles) cur = fetch(unit0);
    for (long long tile = unit0; tile < n_tiles; tile += unit_stride, ++it) {
      const int ab = it & 1;
      const int b = (int)(tile / (p.mt * p.nt)), rem = (int)(tile - (long long)b * p.mt * p.nt);
      const int mi = rem / p.nt, ni = rem % p.nt;
      const int m0 = mi * kUnitM + (int)rank * BM, n0 = ni * BN;
      const int i = m0 + row;                        // row of C
      const bool row_ok = i < p.M;
      // first step: the iterate is the raw Ghat; sigma = q / (||Ghat||_F + eps) is applied here (header)
      const float sig = p.ssq ? sigma_of(cur.tot, p.eps, p.qs) : 1.f;
      // row scalars (E1 needs d_i only on the diagonal tile; rows that need none fetched zeros)
      float d_i = (cur.d0 + cur.d1) * (sig * sig);
      float s_i = 0.f;
      if (EPI == EPI_X && row_ok) s_i = p.a + fmaf(p.beta_h, d_i, cur.s0 + cur.s1);   // a + B_ii, B_ii = beta d_i + (Ah^2)_ii
      if (PAIR) mbar_wait(smem_u32(&ctrl->tfull[ab]), tph[ab]);
      else mbar_wait_parked(smem_u32(&ctrl->tfull[ab]), tph[ab]);
      tph[ab] ^= 1;
      tc_fence_after_sync();
      const Raw nxt = tile + unit_stride < n_tiles ? fetch(tile + unit_stride) : Raw{0.f, 0.f, 0.f, 0.f, 0.f};
      const uint32_t acc = tmem_base + ab * BN + ((uint32_t)(wq * 32) << 16);
      float acc_sq = 0.f;                            // E1: sum_j ACC_ij^2; E3: sum_j x_new_ij^2 over this tile's columns

      if (EPI == EPI_X) {
        const f2 s2 = pk2(s_i, s_i), g2 = pk2(sig, sig);
        f2 sq2 = pk2(0.f, 0.f);
        const uint32_t rs64 = (uint32_t)row * 64u, sw64 = (uint32_t)((row >> 1) & 3);   // 64-byte rows, 64-byte swizzle
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c, ++nchunk) {
          const uint32_t buf = xbuf, par = xpar;
          const uint32_t xs = epi0 + buf * kEpiBuf + rs64;                        // this row of the chunk's hi half
          uint32_t r[16];
          tmem_ld16(acc + 32 * c + 16 * hf, r);
          mbar_wait_parked(smem_u32(&ctrl->xfull[buf]), par);                     // the iterate's chunk has landed
          tmem_wait_ld();
#pragma unroll
          for (int v = 0; v < 2; ++v) {
            const uint32_t a = xs + (((uint32_t)(2 * hf + v) ^ sw64) << 4);
            const uint4 hv = lds128(a), lv = lds128(a + kEpiBuf / 2);
            const uint32_t hw[4] = {hv.x, hv.y, hv.z, hv.w}, lw[4] = {lv.x, lv.y, lv.z, lv.w};
            uint32_t ho[4], lo[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              // x = hi + lo (exact in fp32); x_new = sigma ((a + B_ii) x + ACC); hi' = bf16(x_new), lo' = bf16(x_new - hi')
              const f2 x = pk2(bf16_lo(hw[j]) + bf16_lo(lw[j]), bf16_hi(hw[j]) + bf16_hi(lw[j]));
              const f2 xn = mul2(fma2(s2, x, pk2u(r[8 * v + 2 * j], r[8 * v + 2 * j + 1])), g2);
              sq2 = fma2(xn, xn, sq2);
              float x0, x1;
              upk2(xn, x0, x1);
              ho[j] = pack_bf16(x0, x1);
              lo[j] = pack_bf16(x0 - bf16_lo(ho[j]), x1 - bf16_hi(ho[j]));
            }
            sts128(a, make_uint4(ho[0], ho[1], ho[2], ho[3]));                    // in place
            sts128(a + kEpiBuf / 2, make_uint4(lo[0], lo[1], lo[2], lo[3]));
          }
          fence_proxy_async_smem();
          named_bar_sync(1, kEpiThreads);
          if (et == 0) {
            tma_store_3d(&tmOut, n0 + 32 * c, m0, b, epi0 + buf * kEpiBuf);                 // hi: the next product's operand
            tma_store_3d(&tmLo, n0 + 32 * c, m0, b, epi0 + buf * kEpiBuf + kEpiBuf / 2);
            tma_commit_group();
            // all but this chunk's stores have read their buffers: the PREVIOUS chunk's buffer may be refilled
            tma_wait_group_read1();
            if (nchunk > 0) mbar_arrive(smem_u32(&ctrl->xfree[xprev]));
          }
          xprev = buf;
          if (++xbuf == kXBufs) { xbuf = 0; xpar ^= 1; }
        }
        float q0, q1;
        upk2(sq2, q0, q1);
        acc_sq = q0 + q1;
      } else {
        const float g2s = sig * sig;
        // the accumulator columns of chunk c + 1 are fetched while chunk c is converted, fenced and handed to TMA
        uint32_t rr[2][32];
        tmem_ld32(acc + 32 * hf, rr[0]);
#pragma unroll
        for (int c = 0; c < BN / 64; ++c, ++nchunk) {
          const uint32_t st = epi0 + (nchunk & 1) * kEpiBuf + rsw;                // this row of the [128 x 64] bf16 chunk
          {
            const int hh = hf;
            uint32_t(&r)[32] = rr[c & 1];
            tmem_wait_ld();
            if (c + 1 < BN / 64) tmem_ld32(acc + 64 * (c + 1) + 32 * hh, rr[(c + 1) & 1]);
            if (EPI == EPI_GRAM) {
#pragma unroll
              for (int j = 0; j < 32; ++j) {
                const float v = g2s * __uint_as_float(r[j]);
                r[j] = __float_as_uint(v);
                acc_sq = fmaf(v, v, acc_sq);       // columns beyond N are exact zeros (zero-filled operands)
              }
            }
#pragma unroll
            for (int v = 0; v < 4; ++v) {
              uint4 o;
              o.x = pack_bf16(__uint_as_float(r[8 * v + 0]), __uint_as_float(r[8 * v + 1]));
              o.y = pack_bf16(__uint_as_float(r[8 * v + 2]), __uint_as_float(r[8 * v + 3]));
              o.z = pack_bf16(__uint_as_float(r[8 * v + 4]), __uint_as_float(r[8 * v + 5]));
              o.w = pack_bf16(__uint_as_float(r[8 * v + 6]), __uint_as_float(r[8 * v + 7]));
              sts128(st + ((((uint32_t)(4 * hh + v)) ^ sw) << 4), o);
            }
          }
          // the diagonal of the operand: Ot gets d_i + beta/2 (fp32, rounded once), Bb gets 0
          const int dc = i - (n0 + 64 * c);
          if (row_ok && dc >= 0 && dc < 64 && (dc >> 5) == hf) {   // by the thread that wrote this column
            const __nv_bfloat16 dv = __float2bfloat16_rn(EPI == EPI_GRAM ? fmaf(0.5f, p.beta_h, d_i) : 0.f);
            const uint32_t a = st + ((((uint32_t)(dc >> 3)) ^ sw) << 4) + (uint32_t)(dc & 7) * 2u;
            asm volatile("st.shared.b16 [%0], %1;" ::"r"(a), "h"(*reinterpret_cast<const unsigned short*>(&dv)) : "memory");
          }
          fence_proxy_async_smem();
          // two buffers: the store issued one chunk ago must have read its buffer before anyone passes this barrier and
          // starts writing the next chunk into it (it has had a whole chunk's time to do so)
          if (et == 0) tma_wait_group_read0();
          named_bar_sync(1, kEpiThreads);
          if (et == 0) {
            tma_store_3d(&tmOut, n0 + 64 * c, m0, b, epi0 + (nchunk & 1) * kEpiBuf);
            tma_commit_group();
          }
        }
      }
      tc_fence_before_sync();
      // this thread has read its row of the accumulator
      if (PAIR) mbar_arrive_cluster(mapa_shared(smem_u32(&ctrl->tempty[ab]), 0));
      else mbar_arrive(smem_u32(&ctrl->tempty[ab]));
      if (EPI != EPI_B) {
        // row sums: lower half + upper half, in this order (the next unit's hand-over is behind its chunk barriers)
        if (hf == 1) ctrl->red[row] = acc_sq;
        named_bar_sync(1, kEpiThreads);
        if (hf == 0 && row_ok) {
          const float tot = acc_sq + ctrl->red[row];
          if (EPI == EPI_GRAM) p.s_part[(long long)b * p.ss + (long long)ni * p.rp + i] = tot;
          else p.d_out[(long long)b * p.sd + (long long)ni * p.rp + i] = tot;
        }
      }
      cur = nxt;
    }
    if (et == 0) tma_wait_group0();
  }
  tc_fence_before_sync();
  if (PAIR) {
    cluster_sync_all();
    if (warp == 1) tmem_dealloc_pair<512>(tmem_base);
  } else {
    __syncthreads();
    if (warp == 1) tmem_dealloc<512>(tmem_base);
  }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = [] {
    void* q = nullptr;
    cudaDriverEntryPointQueryResult r;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &q, cudaEnableDefault, &r) != cudaSuccess || r != cudaDriverEntryPointSuccess)
      q = nullptr;
    return reinterpret_cast<EncodeTiledFn>(q);
  }();
  return fn;
}
// [nb][rows][cols] array with row pitch ld and batch pitch sb (elements); box = box_cols x box_rows x 1.
// swizzle: bytes of the swizzle span (128, 64) or 0 for none
bool encode3d(CUtensorMap* out, void* ptr, bool fp32, int cols, int rows, int nb, long long ld, long long sb, int box_cols,
              int box_rows, int swizzle) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  const cuuint64_t es = fp32 ? 4 : 2;
  cuuint64_t dims[3] = {(cuuint64_t)cols, (cuuint64_t)rows, (cuuint64_t)nb};
  cuuint64_t strides[2] = {(cuuint64_t)ld * es, (cuuint64_t)sb * es};
  cuuint32_t box[3] = {(cuuint32_t)box_cols, (cuuint32_t)box_rows, 1u};
  cuuint32_t estr[3] = {1u, 1u, 1u};
  return fn(out, fp32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, ptr, dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : swizzle == 64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_NONE,
            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int EPI, bool B_MN, bool PAIR>
cudaError_t launch_gemm_t(const CUtensorMap& tmA, const CUtensorMap& tmB, const CUtensorMap& tmOut, const CUtensorMap& tmHi,
                          const CUtensorMap& tmLo, GemmParams p, cudaStream_t s) {
  static DeviceOnce once;
  cudaError_t e = configure_smem_once(once, lt_gemm<EPI, B_MN, PAIR>, (int)Cfg<EPI, PAIR>::kSmem);
  if (e != cudaSuccess) return e;
  p.mt = (p.M + (PAIR ? 2 : 1) * BM - 1) / ((PAIR ? 2 : 1) * BM);
  p.nt = (p.N + BN - 1) / BN;
  const long long units = (long long)p.nb * p.mt * p.nt;
  const int ctas = PAIR ? 2 : 1;
  int grid = ctas * (int)std::min<long long>(units, device_sm_count() / ctas);
  if (grid < 1) return cudaSuccess;
  cudaLaunchConfig_t cfg;
  std::memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(kGemmThreads);
  cfg.dynamicSmemBytes = Cfg<EPI, PAIR>::kSmem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = ctas; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, lt_gemm<EPI, B_MN, PAIR>, tmA, tmB, tmOut, tmHi, tmLo, p);
}
// CTA pairs on 256-row blocks when the contraction is long (the full-matrix branch: the mainloop dominates and the
// pair's smaller operand fetch wins, 1.31 -> 1.26 s on the Llama-3-8B shapes); one CTA per 128 x 256 tile otherwise
// (T = 512: eight k-blocks per tile, the pair's cross-CTA hand-overs cost more than its fetch saves, 180 vs 174 ms).
// tmB / tmBp: the B operand's tensor map with the single-CTA box (BN rows) / the pair's (BN / 2 rows per CTA).
template <int EPI, bool B_MN>
cudaError_t launch_gemm(const CUtensorMap& tmA, const CUtensorMap& tmB, const CUtensorMap& tmBp, const CUtensorMap& tmOut,
                        const CUtensorMap& tmHi, const CUtensorMap& tmLo, const GemmParams& p, cudaStream_t s) {
  if (p.M > BM && p.K > 512) return launch_gemm_t<EPI, B_MN, true>(tmA, tmBp, tmOut, tmHi, tmLo, p, s);
  return launch_gemm_t<EPI, B_MN, false>(tmA, tmB, tmOut, tmHi, tmLo, p, s);
}

// One sub-batch of nb tiles of geometry g.
cudaError_t run_sub_batch(const LayerDev* layers_dev, const WorkItem* items_dev, int nb, const LtGeom& g, int whole, int mode,
                          const himuon_hparams& hp, char* scratch, cudaStream_t s, long long* launches) {
  const LtScratch sc = carve(scratch, g, nb);
  const long long sxb = stride_xb(g), sr = stride_r(g), sd = stride_d(g), ssp = stride_s(g);
  const bool step_mode = (mode == MODE_STEP);
  const float qs = sqrtf(sqrtf(hp.c)), beta_h = hp.b / sqrtf(hp.c);
  const dim3 grid_t(kPrepBlocks, nb);
  // big tiles (>= 1 M elements: the full-matrix branch, large rectangular tiles): fused ends on a grid sized by the tile
  // and every TRANSPOSED tile, whatever its size (rectangular tiles taller than wide), through the transposing kernels
  const bool big = (long long)g.rp * g.ldx >= (1ll << 20);
  if (!big && !g.transposed) {
    lt_prep<<<grid_t, kEwThreads, 0, s>>>(layers_dev, items_dev, g, whole, sc.xlo, sc.xb, sxb, sc.d0, sd, sc.ssq,
                                          step_mode ? 1 : 0, hp.beta, hp.nesterov);
    lt_ssq_fold<<<(nb + 255) / 256, 256, 0, s>>>(sc.ssq, nb);
    *launches += 2;
  } else {
    if (g.transposed)
      lt_prep_t<<<dim3((g.rp + kTP - 1) / kTP, g.ntx, nb), kEwThreads, 0, s>>>(layers_dev, items_dev, g, whole, sc.xlo, sc.xb, sxb, sc.d0,
                                                                                sd, step_mode ? 1 : 0, hp.beta, hp.nesterov);
    else
      lt_prep<<<dim3(std::min(1024, (g.rp + 7) / 8), nb), kEwThreads, 0, s>>>(layers_dev, items_dev, g, whole, sc.xlo, sc.xb, sxb, sc.d0, sd,
                                                                               nullptr, step_mode ? 1 : 0, hp.beta, hp.nesterov);
    lt_ssq_from_d<<<nb, 1024, 0, s>>>(sc.d0, sd, g.ntx * g.rp, sc.ssq);
    *launches += 2;
  }
  if (hp.K > 0) {
    // Xb is double-buffered: product 3 of a step reads Xb (all rows of a column block, as the B operand of EVERY row
    // block's tile) while its epilogues write the new Xb, so input and output must be different arrays.
    __nv_bfloat16* xbuf[2] = {sc.xb, sc.xb2};
    CUtensorMap xA[2], xBk[2], xBm[2], xO[2], oA, oB, bA, xL;
    for (int i = 0; i < 2; ++i)
      if (!encode3d(&xA[i], xbuf[i], false, g.np, g.rp, nb, g.ldx, sxb, 64, BM, 128) ||
          !encode3d(&xBk[i], xbuf[i], false, g.np, g.rp, nb, g.ldx, sxb, 64, BN, 128) ||
          !encode3d(&xBm[i], xbuf[i], false, g.np, g.rp, nb, g.ldx, sxb, 64, 64, 128) ||
          !encode3d(&xO[i], xbuf[i], false, g.np, g.rp, nb, g.ldx, sxb, 32, BM, 64))        // E3's 32-column chunks of the iterate's hi half
        return cudaErrorNotSupported;
    if (!encode3d(&oA, sc.ob, false, g.rp, g.rp, nb, g.ldr, sr, 64, BM, 128) ||
        !encode3d(&oB, sc.ob, false, g.rp, g.rp, nb, g.ldr, sr, 64, BN, 128) ||
        !encode3d(&bA, sc.bb, false, g.rp, g.rp, nb, g.ldr, sr, 64, BM, 128) ||
        !encode3d(&xL, sc.xlo, false, g.np, g.rp, nb, g.ldx, sxb, 32, BM, 64))               // ... and of its lo half
      return cudaErrorNotSupported;
    GemmParams p;
    std::memset(&p, 0, sizeof(p));
    p.nb = nb; p.rp = g.rp; p.a = hp.a; p.beta_h = beta_h;
    p.sd = sd; p.ntx = g.ntx; p.ss = ssp; p.ntr = g.ntr; p.s_part = sc.sp;
    p.eps = hp.eps; p.qs = qs;
    float* dcur = sc.d0;
    float* dnext = sc.d1;
    for (int k = 0; k < hp.K; ++k) {
      const int cur = k & 1;
      p.ssq = k == 0 ? sc.ssq : nullptr;         // first step: the iterate is still the raw Ghat
      // A = Xb Xb^T  ->  Ot, S
      p.M = g.rp; p.N = g.rp; p.K = g.np;
      p.d_in = dcur; p.d_out = nullptr;
      cudaError_t e = launch_gemm<EPI_GRAM, false>(xA[cur], xBk[cur], xA[cur], oA, xL, xL, p, s);
      if (e != cudaSuccess) return e;
      // Ot Ot^T  ->  Bb
      p.K = g.rp;
      e = launch_gemm<EPI_B, false>(oA, oB, oA, bA, xL, xL, p, s);
      if (e != cudaSuccess) return e;
      // Bb Xb  ->  new iterate (hi into the other Xb, lo in place), d
      p.M = g.rp; p.N = g.np; p.K = g.rp;
      p.d_out = dnext;
      e = launch_gemm<EPI_X, true>(bA, xBm[cur], xBm[cur], xO[cur ^ 1], xO[cur], xL, p, s);
      if (e != cudaSuccess) return e;
      std::swap(dcur, dnext);
      *launches += 3;
    }
  }
  const __nv_bfloat16* xfin = (hp.K & 1) ? sc.xb2 : sc.xb;
  const float* ssq_fin = hp.K == 0 ? sc.ssq : nullptr;
  if (g.transposed)
    lt_update_t<<<dim3((g.rp + kTP - 1) / kTP, (g.np + kTP - 1) / kTP, nb), kEwThreads, 0, s>>>(
        layers_dev, items_dev, g, whole, xfin, sc.xlo, sxb, step_mode ? 1 : 0, 1.f - hp.lr * hp.wd, -hp.lr * hp.scale_c, 1.f / qs, ssq_fin,
        hp.eps, qs);
  else
    lt_update<<<big ? dim3((unsigned)std::min<long long>(2048, ((long long)g.rp * g.np / 8 + 2 * kEwThreads - 1) / (2 * kEwThreads)), nb) : grid_t,
                kEwThreads, 0, s>>>(layers_dev, items_dev, g, whole, xfin, sc.xlo, sxb, step_mode ? 1 : 0, 1.f - hp.lr * hp.wd,
                                    -hp.lr * hp.scale_c, 1.f / qs, ssq_fin, hp.eps, qs);
  *launches += 1;
  return cudaGetLastError();
}

}  // namespace

size_t lt_path_batch_item_bytes(int Th, int Tw) { return lt_item_bytes(make_geom(Th, Tw)); }
size_t lt_path_scratch_bytes(int h, int w) { return lt_item_bytes(make_geom(h, w)); }

// One chunk of the work list on the large-tile path.  Uniform tiles run in sub-batches of as many tiles as the scratch
// holds; whole-matrix items (T = kWholeMatrixT) run one at a time with the geometry of their own layer.
cudaError_t run_lt_path(const LayerDev* layers_host, const WorkItem* items_host, const LayerDev* layers_dev,
                        const WorkItem* items_dev, long long n_items, int T, int Tw, int mode, const himuon_hparams& hp,
                        void* scratch, size_t scratch_bytes, cudaStream_t s, long long* launches) {
  if (n_items < 1) return cudaSuccess;
  if (T != kWholeMatrixT) {
    const LtGeom g = make_geom(T, Tw);
    const size_t per = lt_item_bytes(g);
    if (scratch_bytes < per) return cudaErrorInvalidValue;
    long long cap = (long long)(scratch_bytes / per);
    if (cap > 65535) cap = 65535;     // the tile index is gridDim.y of the fused ends
    // whole waves: the persistent GEMMs run tiles x CTA-tiles-per-tile work units on one CTA per SM, so a sub-batch whose
    // unit count is a multiple of the SM count has no ragged last wave (T = 512: 4 units per tile, 74 CTA pairs -> 37 tiles)
    {
      const int ctas = (g.rp > BM && g.rp > 512) ? 2 : 1;   // CTA pairs on 256-row blocks when K > 512 (launch_gemm; K = rp in two of three products)
      const long long units = (long long)((g.rp + ctas * BM - 1) / (ctas * BM)) * ((g.np + BN - 1) / BN);
      const long long workers = device_sm_count() / ctas;
      long long a = workers, b = units;
      while (b) { const long long t = a % b; a = b; b = t; }
      const long long wave = workers / a;
      if (cap >= wave) cap -= cap % wave;
    }
    for (long long i = 0; i < n_items; i += cap) {
      const int nb = (int)std::min<long long>(cap, n_items - i);
      cudaError_t e = run_sub_batch(layers_dev, items_dev ? items_dev + i : nullptr, nb, g, items_dev ? 0 : (int)i, mode, hp,
                                    (char*)scratch, s, launches);
      if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
  }
  for (long long i = 0; i < n_items; ++i) {
    const LayerDev& L = layers_host[items_host[i].layer];
    const LtGeom g = make_geom(L.H, L.W);
    if (scratch_bytes < lt_item_bytes(g)) return cudaErrorInvalidValue;
    cudaError_t e = run_sub_batch(layers_dev, items_dev + i, 1, g, 1, mode, hp, (char*)scratch, s, launches);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

}  // namespace himuon
