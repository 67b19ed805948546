// Warp-level tensor-core path of the HiMuon hot path for the small tile sizes T = 16 and T = 32, bf16 storage.
//
// One WARP owns one T x T tile and keeps everything in registers for all K Newton-Schulz steps
// (Eq. 2.2-2.3; nothing between the loads of G, M, W and the stores of M, W touches shared
// or global memory).  Products use mma.sync.m16n8k16 (bf16 operands, fp32 accumulate); the
// accumulator fragment of one product is, after rounding, the A fragment of the next (no data movement),
// the B fragment of a Gram product X X^T is the A fragment of X itself, and the B fragment of B X is the
// A fragment of X transposed 8 x 8 block by block with movmatrix.  These tile sizes are HBM-bound
// (3T flop/B against a ridge of ~250), so the design goal is few instructions per element, not MMA rate.
//
// Numerical scheme = the one of kernels_tc128.cu: fp32 iterate (here: accumulator-layout registers), state
// scaled by c^(1/4) so that B = beta Ah + Ah^2 (beta = b / sqrt(c)); the O(1) diagonal of B never passes
// through bf16 (it acts as the fp32 row scaling a + B_tt); the operand of Ah^2 carries d + beta/2 on its
// diagonal so that offdiag(Ot Ot^T) = offdiag(B).
//
// Fragment layouts (PTX ISA, mma.m16n8k16): g = lane >> 2, c = lane & 3.
//   accumulator of a 16 x 8 block: e = 0,1 -> (row g, col 2c + e); e = 2,3 -> (row g + 8, col 2c + e - 2)
//   A fragment of a 16 x 16 block: a0 (row g, cols 2c..), a1 (row g+8, cols 2c..), a2 (row g, cols 8+2c..),
//                                  a3 (row g+8, cols 8+2c..)
//   B fragment of a 16(k) x 8(n) block: b0 (k = 2c.., n = g), b1 (k = 8+2c.., n = g)
#include <cuda_bf16.h>

#include "himuon_internal.h"

namespace himuon {
namespace {

constexpr int kWarpsPerBlock = 8;
constexpr int kThreads = kWarpsPerBlock * 32;

__device__ __forceinline__ uint32_t pack2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ void mma16816(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t a) {
  uint32_t d;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
  return d;
}
__device__ __forceinline__ float quad_sum(float v) {   // sum over the 4 lanes that share a row
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  return v;
}

// A 16 x 16 block of fp32 values in accumulator layout: v[nh][e], nh = column half (8 columns each).
struct Blk {
  float v[2][4];
};
// ... rounded to bf16 as an A fragment.
__device__ __forceinline__ void to_afrag(const Blk& x, uint32_t (&a)[4]) {
  a[0] = pack2(x.v[0][0], x.v[0][1]);
  a[1] = pack2(x.v[0][2], x.v[0][3]);
  a[2] = pack2(x.v[1][0], x.v[1][1]);
  a[3] = pack2(x.v[1][2], x.v[1][3]);
}

// ... and the bf16 rounding of what the first rounding lost (x - bf16(x)), as a second A fragment.
__device__ __forceinline__ void to_afrag_lo(const Blk& x, const uint32_t (&hi)[4], uint32_t (&lo)[4]) {
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const float a = x.v[r >> 1][2 * (r & 1)], b = x.v[r >> 1][2 * (r & 1) + 1];
    lo[r] = pack2(a - __uint_as_float(hi[r] << 16), b - __uint_as_float(hi[r] & 0xffff0000u));
  }
}

// Accessor of one bf16 matrix tile: element pairs (row, col), (row, col + 1) with col even relative to the
// tile origin.  `fast` = base pointer 4-byte aligned, ld even and the tile origin column even (always: T is
// even), so a pair is one 32-bit access; otherwise two 16-bit accesses.  Out-of-range elements read as zero
// (= the zero padding of B_T) and are not written (= the crop of B_T^-1).
struct TileIO {
  __nv_bfloat16* p;
  long long ld;
  int H, W;      // extent of the matrix
  bool fast;
  __device__ __forceinline__ void load2(int row, int col, float& lo, float& hi) const {
    lo = hi = 0.f;
    if (row >= H || col >= W) return;
    const __nv_bfloat16* q = p + (long long)row * ld + col;
    if (fast && col + 1 < W) {
      const uint32_t u = *reinterpret_cast<const uint32_t*>(q);
      lo = __uint_as_float(u << 16);
      hi = __uint_as_float(u & 0xffff0000u);
    } else {
      lo = __bfloat162float(q[0]);
      if (col + 1 < W) hi = __bfloat162float(q[1]);
    }
  }
  // the same pair as stored bits (lo in the low half), zero outside the matrix
  __device__ __forceinline__ uint32_t load2_raw(int row, int col) const {
    if (row >= H || col >= W) return 0u;
    const __nv_bfloat16* q = p + (long long)row * ld + col;
    if (fast && col + 1 < W) return __ldg(reinterpret_cast<const uint32_t*>(q));
    uint32_t u = *reinterpret_cast<const unsigned short*>(q);
    if (col + 1 < W) u |= (uint32_t)(*reinterpret_cast<const unsigned short*>(q + 1)) << 16;
    return u;
  }
  __device__ __forceinline__ void store2(int row, int col, float lo, float hi) const {
    if (row >= H || col >= W) return;
    __nv_bfloat16* q = p + (long long)row * ld + col;
    if (fast && col + 1 < W) {
      *reinterpret_cast<uint32_t*>(q) = pack2(lo, hi);
    } else {
      q[0] = __float2bfloat16_rn(lo);
      if (col + 1 < W) q[1] = __float2bfloat16_rn(hi);
    }
  }
};
__device__ __forceinline__ TileIO make_io(void* ptr, long long ld, int H, int W) {
  TileIO io;
  io.p = reinterpret_cast<__nv_bfloat16*>(ptr);
  io.ld = ld;
  io.H = H;
  io.W = W;
  io.fast = ((reinterpret_cast<uintptr_t>(ptr) & 3) == 0) && ((ld & 1) == 0);
  return io;
}

// Interior tile with 32-bit-aligned rows: every element pair of the thread is one unchecked 32-bit access at
// base + (2 i + rr) * rows8 + (2 j + nh) * 4 words (base = the thread's first pair, rows8 = 8 rows in words).
struct FastTile {
  bool ok;
  long long g8, m8, w8;         // 8 rows of G / M / W in 32-bit words
  const uint32_t* g;
  uint32_t* m;
  uint32_t* w;
};
__device__ __forceinline__ FastTile make_fast(const LayerDev& L, int row0, int col0, int T, int g, int c, bool step_mode) {
  FastTile f;
  const uintptr_t al = reinterpret_cast<uintptr_t>(L.g) | reinterpret_cast<uintptr_t>(L.w) |
                       (step_mode ? reinterpret_cast<uintptr_t>(L.m) : 0);
  f.ok = (row0 + T <= L.H) && (col0 + T <= L.W) && ((al & 3) == 0) && (((L.ld_g | L.ld_w | (step_mode ? L.ld_m : 0)) & 1) == 0);
  const long long r = row0 + g, cc = col0 + 2 * c;
  f.g = reinterpret_cast<const uint32_t*>(reinterpret_cast<const __nv_bfloat16*>(L.g) + r * L.ld_g + cc);
  f.m = reinterpret_cast<uint32_t*>(reinterpret_cast<__nv_bfloat16*>(L.m) + r * L.ld_m + cc);
  f.w = reinterpret_cast<uint32_t*>(reinterpret_cast<__nv_bfloat16*>(L.w) + r * L.ld_w + cc);
  f.g8 = 4 * L.ld_g;
  f.m8 = 4 * L.ld_m;
  f.w8 = 4 * L.ld_w;
  return f;
}

// The K Newton-Schulz steps on one tile held in registers.  SPLIT: the bf16 operand made from the fp32
// iterate is complemented by the bf16 rounding of its remainder (Gram product with 3 MMAs, B X with 2).
template <int NB, bool SPLIT>
__device__ __forceinline__ void ns_steps(Blk (&x)[NB][NB], float (&d)[NB][2], const himuon_hparams& hp, float beta_h,
                                         bool pd0, bool pd1) {
#pragma unroll 1
  for (int k = 0; k < hp.K; ++k) {
    uint32_t xa[NB][NB][4], xl[SPLIT ? NB : 1][SPLIT ? NB : 1][4];
#pragma unroll
    for (int i = 0; i < NB; ++i)
#pragma unroll
      for (int j = 0; j < NB; ++j) {
        to_afrag(x[i][j], xa[i][j]);
        if (SPLIT) to_afrag_lo(x[i][j], xa[i][j], xl[SPLIT ? i : 0][SPLIT ? j : 0]);
      }

    // Ah = Xb Xb^T
    Blk A[NB][NB];
#pragma unroll
    for (int i = 0; i < NB; ++i)
#pragma unroll
      for (int j = 0; j < NB; ++j)
#pragma unroll
        for (int nh = 0; nh < 2; ++nh) {
#pragma unroll
          for (int e = 0; e < 4; ++e) A[i][j].v[nh][e] = 0.f;
#pragma unroll
          for (int kb = 0; kb < NB; ++kb) {
            mma16816(A[i][j].v[nh], xa[i][kb], xa[j][kb][nh], xa[j][kb][nh + 2]);
            if (SPLIT) {   // (Xh + Xl)(Xh + Xl)^T without the Xl Xl^T term
              mma16816(A[i][j].v[nh], xa[i][kb], xl[SPLIT ? j : 0][SPLIT ? kb : 0][nh], xl[SPLIT ? j : 0][SPLIT ? kb : 0][nh + 2]);
              mma16816(A[i][j].v[nh], xl[SPLIT ? i : 0][SPLIT ? kb : 0], xa[j][kb][nh], xa[j][kb][nh + 2]);
            }
          }
        }
    // a + B_tt with B_tt = beta d_t + (Ah^2)_tt, (Ah^2)_tt = sum_j Ah_tj^2: fp32 row scaling
    float si[NB][2];
#pragma unroll
    for (int i = 0; i < NB; ++i) {
      float p0 = 0.f, p1 = 0.f;
#pragma unroll
      for (int j = 0; j < NB; ++j)
#pragma unroll
        for (int nh = 0; nh < 2; ++nh) {
          p0 = fmaf(A[i][j].v[nh][0], A[i][j].v[nh][0], fmaf(A[i][j].v[nh][1], A[i][j].v[nh][1], p0));
          p1 = fmaf(A[i][j].v[nh][2], A[i][j].v[nh][2], fmaf(A[i][j].v[nh][3], A[i][j].v[nh][3], p1));
        }
      si[i][0] = hp.a + fmaf(beta_h, d[i][0], quad_sum(p0));
      si[i][1] = hp.a + fmaf(beta_h, d[i][1], quad_sum(p1));
      // Ot = offdiag(Ah) + diag(d + beta/2): offdiag(Ot Ot^T) = offdiag(beta Ah + Ah^2)
      const float dv0 = fmaf(0.5f, beta_h, d[i][0]), dv1 = fmaf(0.5f, beta_h, d[i][1]);
      if (pd0) { A[i][i].v[0][0] = dv0; A[i][i].v[1][2] = dv1; }
      if (pd1) { A[i][i].v[0][1] = dv0; A[i][i].v[1][3] = dv1; }
    }
    uint32_t oa[NB][NB][4];
#pragma unroll
    for (int i = 0; i < NB; ++i)
#pragma unroll
      for (int j = 0; j < NB; ++j) to_afrag(A[i][j], oa[i][j]);

    // B (off the diagonal) = Ot Ot^T, rounded to bf16 with the diagonal zeroed
    uint32_t ba[NB][NB][4];
#pragma unroll
    for (int i = 0; i < NB; ++i)
#pragma unroll
      for (int j = 0; j < NB; ++j) {
        Blk Bm;
#pragma unroll
        for (int nh = 0; nh < 2; ++nh) {
#pragma unroll
          for (int e = 0; e < 4; ++e) Bm.v[nh][e] = 0.f;
#pragma unroll
          for (int kb = 0; kb < NB; ++kb) mma16816(Bm.v[nh], oa[i][kb], oa[j][kb][nh], oa[j][kb][nh + 2]);
        }
        if (i == j) {
          if (pd0) { Bm.v[0][0] = 0.f; Bm.v[1][2] = 0.f; }
          if (pd1) { Bm.v[0][1] = 0.f; Bm.v[1][3] = 0.f; }
        }
        to_afrag(Bm, ba[i][j]);
      }

    // Xh <- (a + B_tt) Xh + offdiag(B) Xb: scale the state, then accumulate the product onto it
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      uint32_t xt[NB][2][2], xtl[SPLIT ? NB : 1][2][2];   // B fragments of Xb(kb, j): [kb][nh][b0 / b1]
#pragma unroll
      for (int kb = 0; kb < NB; ++kb) {
        xt[kb][0][0] = movmatrix_trans(xa[kb][j][0]);
        xt[kb][0][1] = movmatrix_trans(xa[kb][j][1]);
        xt[kb][1][0] = movmatrix_trans(xa[kb][j][2]);
        xt[kb][1][1] = movmatrix_trans(xa[kb][j][3]);
        if (SPLIT) {
          xtl[SPLIT ? kb : 0][0][0] = movmatrix_trans(xl[SPLIT ? kb : 0][SPLIT ? j : 0][0]);
          xtl[SPLIT ? kb : 0][0][1] = movmatrix_trans(xl[SPLIT ? kb : 0][SPLIT ? j : 0][1]);
          xtl[SPLIT ? kb : 0][1][0] = movmatrix_trans(xl[SPLIT ? kb : 0][SPLIT ? j : 0][2]);
          xtl[SPLIT ? kb : 0][1][1] = movmatrix_trans(xl[SPLIT ? kb : 0][SPLIT ? j : 0][3]);
        }
      }
#pragma unroll
      for (int i = 0; i < NB; ++i)
#pragma unroll
        for (int nh = 0; nh < 2; ++nh) {
          x[i][j].v[nh][0] *= si[i][0];
          x[i][j].v[nh][1] *= si[i][0];
          x[i][j].v[nh][2] *= si[i][1];
          x[i][j].v[nh][3] *= si[i][1];
#pragma unroll
          for (int kb = 0; kb < NB; ++kb) {
            mma16816(x[i][j].v[nh], ba[i][kb], xt[kb][nh][0], xt[kb][nh][1]);
            if (SPLIT) mma16816(x[i][j].v[nh], ba[i][kb], xtl[SPLIT ? kb : 0][nh][0], xtl[SPLIT ? kb : 0][nh][1]);
          }
        }
    }
    if (k + 1 < hp.K) {
#pragma unroll
      for (int i = 0; i < NB; ++i) {
        float p0 = 0.f, p1 = 0.f;
#pragma unroll
        for (int j = 0; j < NB; ++j)
#pragma unroll
          for (int nh = 0; nh < 2; ++nh) {
            p0 = fmaf(x[i][j].v[nh][0], x[i][j].v[nh][0], fmaf(x[i][j].v[nh][1], x[i][j].v[nh][1], p0));
            p1 = fmaf(x[i][j].v[nh][2], x[i][j].v[nh][2], fmaf(x[i][j].v[nh][3], x[i][j].v[nh][3], p1));
          }
        d[i][0] = quad_sum(p0);
        d[i][1] = quad_sum(p1);
      }
    }
  }
}

template <int NB>
__global__ void __launch_bounds__(kThreads)
himuon_warp_kernel(const LayerDev* __restrict__ layers, const WorkItem* __restrict__ items, long long n_items,
                   int mode, himuon_hparams hp) {
  constexpr int T = 16 * NB;
  const int lane = threadIdx.x & 31, g = lane >> 2, c = lane & 3;
  const bool step_mode = (mode == MODE_STEP);
  // the diagonal element of row g (and of row g + 8) of a diagonal 16 x 16 block sits in lane c == g >> 1,
  // accumulator slot e = g & 1 of column half 0 (slot 2 + (g & 1) of column half 1)
  const bool pd0 = (c == (g >> 1)) && !(g & 1), pd1 = (c == (g >> 1)) && (g & 1);
  const float qs = sqrtf(sqrtf(hp.c));          // state Xh = c^(1/4) X, see kernels_tc128.cu
  const float beta_h = hp.b / sqrtf(hp.c);
  const long long stride = (long long)gridDim.x * kWarpsPerBlock;

  // Software pipeline over the warp's tiles: the work item, the layer descriptor and the raw G / M bits of
  // the NEXT tile are requested before the Newton-Schulz steps of the current one, and W of the current
  // tile before its steps, so that the dependent chain item -> layer -> data never stalls the warp.
  auto fetch = [&](long long i, LayerDev& L, int& row0, int& col0, uint32_t (&gq)[NB * NB * 4], uint32_t (&mq)[NB * NB * 4]) {
    WorkItem wi;
    if (items) wi = items[i];
    else { wi.layer = 0; wi.r = (int)i; wi.c = 0; wi.pad = 0; }
    L = layers[wi.layer];
    row0 = wi.r * T;
    col0 = wi.c * T;
    const FastTile ft = make_fast(L, row0, col0, T, g, c, step_mode);
    if (ft.ok) {
#pragma unroll
      for (int q = 0; q < NB * NB * 4; ++q) {
        const int i2 = q / (NB * 4), j2 = (q / 4) % NB, nh = (q >> 1) & 1, rr = q & 1;
        gq[q] = __ldg(ft.g + (2 * i2 + rr) * ft.g8 + (2 * j2 + nh) * 4);
        mq[q] = step_mode ? ft.m[(2 * i2 + rr) * ft.m8 + (2 * j2 + nh) * 4] : 0u;
      }
      return;
    }
    const TileIO ioG = make_io(L.g, L.ld_g, L.H, L.W);
    const TileIO ioM = make_io(L.m, L.ld_m, L.H, L.W);
#pragma unroll
    for (int q = 0; q < NB * NB * 4; ++q) {
      const int i2 = q / (NB * 4), j2 = (q / 4) % NB, nh = (q >> 1) & 1, rr = q & 1;
      const int row = row0 + 16 * i2 + g + 8 * rr, col = col0 + 16 * j2 + 8 * nh + 2 * c;
      gq[q] = ioG.load2_raw(row, col);
      mq[q] = step_mode ? ioM.load2_raw(row, col) : 0u;
    }
  };

  long long it = (long long)blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
  LayerDev Ln;
  int rown = 0, coln = 0;
  uint32_t gq[NB * NB * 4], mq[NB * NB * 4];
  if (it < n_items) fetch(it, Ln, rown, coln, gq, mq);

  while (it < n_items) {
    const LayerDev L = Ln;
    const int row0 = rown, col0 = coln;
    const TileIO ioM = make_io(L.m, L.ld_m, L.H, L.W);
    const TileIO ioW = make_io(L.w, L.ld_w, L.H, L.W);
    const FastTile ft = make_fast(L, row0, col0, T, g, c, step_mode);

    // ---------------- P: momentum, Frobenius normalisation ----------
    Blk x[NB][NB];
    float ss = 0.f;
#pragma unroll
    for (int q = 0; q < NB * NB * 4; ++q) {
      const int i = q / (NB * 4), j = (q / 4) % NB, nh = (q >> 1) & 1, rr = q & 1;
      const int row = row0 + 16 * i + g + 8 * rr, col = col0 + 16 * j + 8 * nh + 2 * c;
      const float g0 = __uint_as_float(gq[q] << 16), g1 = __uint_as_float(gq[q] & 0xffff0000u);
      float h0 = g0, h1 = g1;
      if (step_mode) {
        const float m0 = fmaf(hp.beta, __uint_as_float(mq[q] << 16), g0);
        const float m1 = fmaf(hp.beta, __uint_as_float(mq[q] & 0xffff0000u), g1);
        if (ft.ok) ft.m[(2 * i + rr) * ft.m8 + (2 * j + nh) * 4] = pack2(m0, m1);
        else ioM.store2(row, col, m0, m1);
        h0 = hp.nesterov ? fmaf(hp.beta, m0, g0) : m0;     // Ghat = G + beta M' (Nesterov) | M'
        h1 = hp.nesterov ? fmaf(hp.beta, m1, g1) : m1;
      }
      x[i][j].v[nh][2 * rr] = h0;
      x[i][j].v[nh][2 * rr + 1] = h1;
      ss = fmaf(h0, h0, fmaf(h1, h1, ss));
    }
    const long long nx = it + stride;
    if (nx < n_items) fetch(nx, Ln, rown, coln, gq, mq);      // consumed in the next iteration
    uint32_t wq[NB * NB * 4];                                  // W of this tile, consumed after the steps
#pragma unroll
    for (int q = 0; q < NB * NB * 4; ++q) {
      const int i = q / (NB * 4), j = (q / 4) % NB, nh = (q >> 1) & 1, rr = q & 1;
      if (!step_mode) wq[q] = 0u;
      else if (ft.ok) wq[q] = ft.w[(2 * i + rr) * ft.w8 + (2 * j + nh) * 4];
      else wq[q] = ioW.load2_raw(row0 + 16 * i + g + 8 * rr, col0 + 16 * j + 8 * nh + 2 * c);
    }
    float tot = ss;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
    const float nrm = sqrtf(tot);
    const float inv = nrm > 0.f ? qs / (nrm + hp.eps) : 0.f;   // Phi_K(0) = 0
    float d[NB][2];                                             // d = diag(Ah) in fp32, rows g / g + 8 of block row i
#pragma unroll
    for (int i = 0; i < NB; ++i) {
      float p0 = 0.f, p1 = 0.f;
#pragma unroll
      for (int j = 0; j < NB; ++j)
#pragma unroll
        for (int nh = 0; nh < 2; ++nh)
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const float v = x[i][j].v[nh][e] * inv;
            x[i][j].v[nh][e] = v;
            if (e < 2) p0 = fmaf(v, v, p0); else p1 = fmaf(v, v, p1);
          }
      d[i][0] = quad_sum(p0);
      d[i][1] = quad_sum(p1);
    }

    // ---------------- K Newton-Schulz steps -------------------------------------------
    // Ragged edge tiles have few rows or columns and so few singular directions to average rounding errors
    // over; they run with the iterate split into bf16 hi + lo parts (errors ~4x smaller, 2x the MMAs).
    const bool ragged = (row0 + T > L.H) || (col0 + T > L.W);
    if (ragged) ns_steps<NB, true>(x, d, hp, beta_h, pd0, pd1);
    else ns_steps<NB, false>(x, d, hp, beta_h, pd0, pd1);

    // ---------------- F: untile + scaled, weight-decayed write (Eq. 4.6) ---------------
    const float keep = 1.f - hp.lr * hp.wd;
    const float unq = 1.f / qs;
    const float stepsz = step_mode ? -hp.lr * hp.scale_c * L.tau_base * unq : unq;
#pragma unroll
    for (int q = 0; q < NB * NB * 4; ++q) {
      const int i = q / (NB * 4), j = (q / 4) % NB, nh = (q >> 1) & 1, rr = q & 1;
      const int row = row0 + 16 * i + g + 8 * rr, col = col0 + 16 * j + 8 * nh + 2 * c;
      float o0 = stepsz * x[i][j].v[nh][2 * rr], o1 = stepsz * x[i][j].v[nh][2 * rr + 1];
      if (step_mode) {
        o0 = fmaf(keep, __uint_as_float(wq[q] << 16), o0);
        o1 = fmaf(keep, __uint_as_float(wq[q] & 0xffff0000u), o1);
      }
      if (ft.ok) ft.w[(2 * i + rr) * ft.w8 + (2 * j + nh) * 4] = pack2(o0, o1);
      else ioW.store2(row, col, o0, o1);
    }
    it = nx;
  }
}

}  // namespace

cudaError_t launch_warp(const LaunchArgs& a, cudaStream_t s) {
  if (a.n_items < 1) return cudaSuccess;
  long long grid = (a.n_items + kWarpsPerBlock - 1) / kWarpsPerBlock;
  const long long cap = (long long)device_sm_count() * 8;
  if (grid > cap) grid = cap;
  if (a.T == 16) himuon_warp_kernel<1><<<(unsigned)grid, kThreads, 0, s>>>(a.layers, a.items, a.n_items, a.mode, a.hp);
  else if (a.T == 32) himuon_warp_kernel<2><<<(unsigned)grid, kThreads, 0, s>>>(a.layers, a.items, a.n_items, a.mode, a.hp);
  else return cudaErrorInvalidValue;
  return cudaGetLastError();
}

}  // namespace himuon
