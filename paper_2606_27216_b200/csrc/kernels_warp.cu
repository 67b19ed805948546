// Warp-level tensor-core path of the HiMuon hot path for the small tile sizes T = 16 and T = 32, bf16 storage.
//
// One WARP owns one T x T tile and keeps the fp32 iterate in registers for all K Newton-Schulz steps
// (Eq. 2.2-2.3; nothing between the loads of G, M, W and the stores of M, W touches global memory,
// PAPER.md:221).  These tile sizes are HBM-bound (3T flop/B against a ridge of ~250), so the design goals are
// (1) full-width memory transactions and a deep prefetch, (2) few instructions per element:
//
//   * Column relabelling.  Phi_K(X P) = Phi_K(X) P for a permutation P, so WHICH columns of the tile a lane holds is
//     free as long as load and store agree.  Lane (g, c) (g = lane >> 2, c = lane & 3) holds, of rows g and g + 8 of
//     every 16-row block, the T/4 CONSECUTIVE columns c T/4 .. : one 8-byte (T = 16) or 16-byte (T = 32) access per
//     row, a warp instruction covers whole rows, every 32-byte sector is used in full.
//   * G, M, W of the NEXT tile stream into a warp-private shared-memory buffer with cp.async while the current
//     tile's steps run (each lane copies exactly the bytes it reads back, so no barrier is involved).
//   * A = X X^T and A^2 = A A^T are tf32 mma.sync.m16n8k8 products straight out of the fp32 accumulator-layout
//     registers: with the k index relabelled (k = c <-> column 2c, k = c + 4 <-> column 2c + 1) the accumulator
//     fragment of one product IS the A fragment and (for these X X^T-form products) the B fragment of the next, no
//     data movement, no packing.  tf32 keeps the O(1) diagonals of A and B to 2^-11, so the polynomial
//     B = b A + c A^2 is formed in plain fp32 and its diagonal acts as the fp32 row scaling a + B_tt - no scaled
//     state, no operand-diagonal trick, no row-sum reductions (and any finite (a, b, c) works).
//   * X <- (a + B_tt) X + offdiag(B) X needs X as a [k][n] operand, i.e. transposed across lanes: that product runs
//     as bf16 mma.sync.m16n8k16 with the B fragment made by movmatrix (8 x 8 b16 transposes) from the packed iterate.
// Measured per-tile error against the float64 oracle: see DESIGN.md section 5.
//
// Fragment layouts (PTX ISA), g = lane >> 2, c = lane & 3:
//   accumulator of a 16 x 8 block (both shapes): e = 0,1 -> (row g, col 2c + e); e = 2,3 -> (row g + 8, col 2c + e - 2)
//   m16n8k8 tf32:   A: a0 (g, k=c) a1 (g+8, k=c) a2 (g, k=c+4) a3 (g+8, k=c+4);   B: b0 (k=c, n=g) b1 (k=c+4, n=g)
//   m16n8k16 bf16:  A: a0 (g, 2c..) a1 (g+8, 2c..) a2 (g, 8+2c..) a3 (g+8, 8+2c..);  B: b0 (k=2c.., n=g) b1 (k=8+2c.., n=g)
#include <cuda_bf16.h>

#include <type_traits>

#include "himuon_internal.h"

namespace himuon {
namespace {

// T = 16: blocks of 8 warps, 4 per SM (64 registers).  T = 32: the three 32 x 32 fp32 matrices of a step (X, A, B) are 96
// registers of a lane, so blocks of 4 warps, 3 per SM (168 registers, no spills; at 128 registers the step spills).
template <int NB> struct Cfg {
  static constexpr int kWarps = NB == 1 ? 8 : 4;
  static constexpr int kBlocksPerSm = NB == 1 ? 4 : 3;
};

__device__ __forceinline__ uint32_t pack2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ float bf_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf_hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }
// fp32 -> tf32, round to nearest (ties away): the tensor core ignores the 13 low mantissa bits, so adding half of the
// tf32 spacing to the bit pattern IS the rounding - one integer add.  (cvt.rna.tf32.f32 compiles to this add plus an
// Inf / NaN guard, three instructions per value; the iterate and its Gram matrices are bounded by ~1.2.)
__device__ __forceinline__ uint32_t to_tf32(float x) { return __float_as_uint(x) + 0x1000u; }
__device__ __forceinline__ void mma_tf32(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void mma_bf16(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t a) {
  uint32_t d;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
  return d;
}
template <int kBytes>
__device__ __forceinline__ void cp_async(uint32_t dst_smem, const void* src) {
  if constexpr (kBytes == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst_smem), "l"(src) : "memory");
  else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst_smem), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// A 16 x 16 block in accumulator layout: v[h][e], h = 8-column half, e as above (fp32 values or tf32 bit patterns).
struct Blk {
  float v[2][4];
};
struct BlkU {
  uint32_t v[2][4];
};

// D (+)= P Q^T for 16 x 16 blocks held in accumulator layout (tf32 bit patterns): k-slice (kh) of P as the A fragment,
// rows 8 nn + g of Q as the B fragment - all operands are the lane's own registers.
__device__ __forceinline__ void gram_block(Blk& d, const BlkU& p, const BlkU& q) {
#pragma unroll
  for (int nn = 0; nn < 2; ++nn)
#pragma unroll
    for (int kh = 0; kh < 2; ++kh)
      mma_tf32(d.v[nn], p.v[kh][0], p.v[kh][2], p.v[kh][1], p.v[kh][3], q.v[kh][2 * nn], q.v[kh][2 * nn + 1]);
}

template <int NB>
__global__ void __launch_bounds__(Cfg<NB>::kWarps * 32, Cfg<NB>::kBlocksPerSm)
himuon_warp_kernel(const LayerDev* __restrict__ layers, const WorkItem* __restrict__ items, long long n_items,
                   int mode, himuon_hparams hp) {
  constexpr int T = 16 * NB;
  constexpr int kWarpsPerBlock = Cfg<NB>::kWarps;
  constexpr int kLaneBytes = T / 2;                // bytes of a row held by one lane: 8 (T = 16) / 16 (T = 32)
  constexpr int kRowBytes = 2 * T;
  constexpr int kTileBytes = T * kRowBytes;
  constexpr int kRowsPerLane = 2 * NB;             // rows 16 i + g and 16 i + g + 8
  typedef typename std::conditional<NB == 1, uint2, uint4>::type vec_t;   // one lane's share of a row
  extern __shared__ __align__(16) uint8_t smem[];
  const int lane = threadIdx.x & 31, g = lane >> 2, c = lane & 3, warp = threadIdx.x >> 5;
  const bool step_mode = (mode == MODE_STEP);
  // the diagonal element of row g (and of row g + 8) of a diagonal 16 x 16 block sits in lane c == g >> 1,
  // accumulator slot e = g & 1 of column half 0 (slot 2 + (g & 1) of column half 1)
  const bool pd = (c == (g >> 1));
  const int pe = g & 1;
  const int diag_src = (lane & ~3) | (g >> 1);
  const long long stride = (long long)gridDim.x * kWarpsPerBlock;
  // warp-private staging: 2 buffers x (G, M, W); a lane's bytes of row r: r * kRowBytes + c * kLaneBytes
  const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem) + warp * (2 * 3 * kTileBytes);
  const uint32_t lane_off = (uint32_t)g * kRowBytes + (uint32_t)c * kLaneBytes;

  struct TileAt {
    const uint8_t *pg;
    uint8_t *pm, *pw;         // this lane's first element (row g of the tile, its column group)
    long long sg, sm, sw;     // row strides in bytes
    int rows, cols;           // live extent of the tile
    float tau_base;
    bool fast;                // interior tile, aligned: vector accesses without bounds checks
  };
  auto locate = [&](long long i) {
    WorkItem wi;
    if (items) wi = items[i];
    else { wi.layer = 0; wi.r = (int)i; wi.c = 0; wi.pad = 0; }
    const LayerDev L = layers[wi.layer];
    TileAt t;
    const long long row0 = (long long)wi.r * T, col0 = (long long)wi.c * T;
    t.rows = (int)min((long long)T, L.H - row0);
    t.cols = (int)min((long long)T, L.W - col0);
    t.sg = L.ld_g * 2; t.sm = L.ld_m * 2; t.sw = L.ld_w * 2;
    const long long col = col0 + c * (T / 4);
    t.pg = reinterpret_cast<const uint8_t*>(L.g) + (row0 + g) * t.sg + col * 2;
    t.pm = L.m ? reinterpret_cast<uint8_t*>(L.m) + (row0 + g) * t.sm + col * 2 : nullptr;
    t.pw = reinterpret_cast<uint8_t*>(L.w) + (row0 + g) * t.sw + col * 2;
    const uintptr_t al = reinterpret_cast<uintptr_t>(L.g) | reinterpret_cast<uintptr_t>(L.w) | (uintptr_t)t.sg | (uintptr_t)t.sw |
                         (step_mode ? (reinterpret_cast<uintptr_t>(L.m) | (uintptr_t)t.sm) : 0);
    t.fast = (t.rows == T) && (t.cols == T) && ((al & (kLaneBytes - 1)) == 0);
    t.tau_base = L.tau_base;
    return t;
  };
  // stream a tile's G, M (and W) into staging buffer `buf` (fast tiles only; others are read directly when needed)
  auto prefetch = [&](const TileAt& t, int buf) {
    if (!t.fast) return;
    const uint32_t dst = sbase + buf * (3 * kTileBytes) + lane_off;
#pragma unroll
    for (int r = 0; r < kRowsPerLane; ++r) {
      cp_async<kLaneBytes>(dst + r * 8 * kRowBytes, t.pg + (long long)r * 8 * t.sg);
      if (step_mode) {
        cp_async<kLaneBytes>(dst + kTileBytes + r * 8 * kRowBytes, t.pm + (long long)r * 8 * t.sm);
        cp_async<kLaneBytes>(dst + 2 * kTileBytes + r * 8 * kRowBytes, t.pw + (long long)r * 8 * t.sw);
      }
    }
  };
  // one lane's share of row r (0 .. 2 NB - 1 -> tile row g + 8 r) of a tensor: staging buffer (fast) or global memory
  auto read_row = [&](const TileAt& t, int buf, int which, const uint8_t* gp, long long gs, int r, uint32_t (&w)[kLaneBytes / 4]) {
    if (t.fast) {
      const uint32_t a = sbase + buf * (3 * kTileBytes) + which * kTileBytes + lane_off + r * 8 * kRowBytes;
      if constexpr (NB == 1) asm volatile("ld.shared.v2.b32 {%0, %1}, [%2];" : "=r"(w[0]), "=r"(w[1]) : "r"(a));
      else asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]) : "r"(a));
    } else {   // edge or unaligned tile: element by element, zero outside the matrix (B_T padding)
      const unsigned short* p = reinterpret_cast<const unsigned short*>(gp + (long long)r * 8 * gs);
      const int row = g + 8 * r;
#pragma unroll
      for (int q = 0; q < kLaneBytes / 4; ++q) {
        const int col = c * (T / 4) + 2 * q;
        uint32_t lo = 0, hi = 0;
        if (gp && row < t.rows) {
          if (col < t.cols) lo = p[2 * q];
          if (col + 1 < t.cols) hi = p[2 * q + 1];
        }
        w[q] = lo | (hi << 16);
      }
    }
  };
  auto write_row = [&](const TileAt& t, uint8_t* gp, long long gs, int r, const uint32_t (&w)[kLaneBytes / 4]) {
    if (t.fast) {
      vec_t v;
      if constexpr (NB == 1) v = make_uint2(w[0], w[1]);
      else v = make_uint4(w[0], w[1], w[2], w[3]);
      *reinterpret_cast<vec_t*>(gp + (long long)r * 8 * gs) = v;
    } else {   // crop of B_T^-1
      unsigned short* p = reinterpret_cast<unsigned short*>(gp + (long long)r * 8 * gs);
      const int row = g + 8 * r;
#pragma unroll
      for (int q = 0; q < kLaneBytes / 4; ++q) {
        const int col = c * (T / 4) + 2 * q;
        if (row < t.rows) {
          if (col < t.cols) p[2 * q] = (unsigned short)(w[q] & 0xffffu);
          if (col + 1 < t.cols) p[2 * q + 1] = (unsigned short)(w[q] >> 16);
        }
      }
    }
  };
  // Register home of a lane's 4 consecutive columns of 16-column block j, rows g (rr = 0) / g + 8 (rr = 1) of block row i:
  // x[i][j].v[0][2 rr + {0,1}], x[i][j].v[1][2 rr + {0,1}].  Word q of the lane's row share = columns 2q, 2q + 1 of its
  // group: block j = q / 2, half h = q % 2.

  long long it = (long long)blockIdx.x * kWarpsPerBlock + warp;
  TileAt cur;
  int buf = 0;
  if (it < n_items) {
    cur = locate(it);
    prefetch(cur, 0);
  }
  cp_async_commit();

  while (it < n_items) {
    const long long nx = it + stride;
    TileAt nxt = cur;
    cp_async_wait_all();                 // this tile's G, M, W are in the staging buffer
    if (nx < n_items) {
      nxt = locate(nx);
      prefetch(nxt, buf ^ 1);            // in flight during this tile's steps
    }
    cp_async_commit();

    // ---------------- P: momentum, Frobenius normalisation ----------
    Blk x[NB][NB];
    float ss = 0.f;
#pragma unroll
    for (int r = 0; r < kRowsPerLane; ++r) {
      const int i = r >> 1, rr = r & 1;
      uint32_t gw[kLaneBytes / 4], mw[kLaneBytes / 4], mo[kLaneBytes / 4];
      read_row(cur, buf, 0, cur.pg, cur.sg, r, gw);
      if (step_mode) read_row(cur, buf, 1, cur.pm, cur.sm, r, mw);
#pragma unroll
      for (int q = 0; q < kLaneBytes / 4; ++q) {
        const float g0 = bf_lo(gw[q]), g1 = bf_hi(gw[q]);
        float h0 = g0, h1 = g1;
        if (step_mode) {
          const float m0 = fmaf(hp.beta, bf_lo(mw[q]), g0), m1 = fmaf(hp.beta, bf_hi(mw[q]), g1);
          mo[q] = pack2(m0, m1);
          h0 = hp.nesterov ? fmaf(hp.beta, m0, g0) : m0;     // Ghat = G + beta M' (Nesterov) | M'
          h1 = hp.nesterov ? fmaf(hp.beta, m1, g1) : m1;
        }
        x[i][q >> 1].v[q & 1][2 * rr] = h0;
        x[i][q >> 1].v[q & 1][2 * rr + 1] = h1;
        ss = fmaf(h0, h0, fmaf(h1, h1, ss));
      }
      if (step_mode) write_row(cur, cur.pm, cur.sm, r, mo);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
    const float nrm = sqrtf(ss);
    const float inv = nrm > 0.f ? 1.f / (nrm + hp.eps) : 0.f;   // Phi_K(0) = 0
#pragma unroll
    for (int i = 0; i < NB; ++i)
#pragma unroll
      for (int j = 0; j < NB; ++j)
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
          for (int e = 0; e < 4; ++e) x[i][j].v[h][e] *= inv;

    // ---------------- K Newton-Schulz steps -------------------------------------------
#pragma unroll 1
    for (int k = 0; k < hp.K; ++k) {
      // A = X X^T (tf32)
      Blk A[NB][NB];
      {
        BlkU xt[NB][NB];
#pragma unroll
        for (int i = 0; i < NB; ++i)
#pragma unroll
          for (int j = 0; j < NB; ++j)
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
              for (int e = 0; e < 4; ++e) xt[i][j].v[h][e] = to_tf32(x[i][j].v[h][e]);
#pragma unroll
        for (int i = 0; i < NB; ++i)
#pragma unroll
          for (int j = 0; j < NB; ++j) {
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
              for (int e = 0; e < 4; ++e) A[i][j].v[h][e] = 0.f;
#pragma unroll
            for (int kb = 0; kb < NB; ++kb) gram_block(A[i][j], xt[i][kb], xt[j][kb]);
          }
      }
      // B = b A + c A^2 (A symmetric: A^2 = A A^T, the same register-only product form)
      Blk Bm[NB][NB];
      {
        BlkU at[NB][NB];
#pragma unroll
        for (int i = 0; i < NB; ++i)
#pragma unroll
          for (int j = 0; j < NB; ++j)
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
              for (int e = 0; e < 4; ++e) at[i][j].v[h][e] = to_tf32(A[i][j].v[h][e]);
#pragma unroll
        for (int i = 0; i < NB; ++i)
#pragma unroll
          for (int j = 0; j < NB; ++j) {
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
              for (int e = 0; e < 4; ++e) Bm[i][j].v[h][e] = 0.f;
#pragma unroll
            for (int kb = 0; kb < NB; ++kb) gram_block(Bm[i][j], at[i][kb], at[j][kb]);
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
              for (int e = 0; e < 4; ++e) Bm[i][j].v[h][e] = fmaf(hp.c, Bm[i][j].v[h][e], hp.b * A[i][j].v[h][e]);
          }
      }
      // a + B_tt as an fp32 row scaling; the diagonal leaves the bf16 operand
      float s0[NB], s1[NB];
#pragma unroll
      for (int i = 0; i < NB; ++i) {
        const float d0 = pe ? Bm[i][i].v[0][1] : Bm[i][i].v[0][0];      // (g, g) where this lane holds it
        const float d1 = pe ? Bm[i][i].v[1][3] : Bm[i][i].v[1][2];      // (g + 8, g + 8)
        s0[i] = hp.a + __shfl_sync(0xffffffffu, d0, diag_src);
        s1[i] = hp.a + __shfl_sync(0xffffffffu, d1, diag_src);
        if (pd) {
          if (pe) { Bm[i][i].v[0][1] = 0.f; Bm[i][i].v[1][3] = 0.f; }
          else { Bm[i][i].v[0][0] = 0.f; Bm[i][i].v[1][2] = 0.f; }
        }
      }
      // X <- (a + B_tt) X + offdiag(B) Xb   (bf16 m16n8k16; B fragment of Xb by movmatrix)
      uint32_t ba[NB][NB][4], xa[NB][NB][4];
#pragma unroll
      for (int i = 0; i < NB; ++i)
#pragma unroll
        for (int j = 0; j < NB; ++j) {
          ba[i][j][0] = pack2(Bm[i][j].v[0][0], Bm[i][j].v[0][1]);
          ba[i][j][1] = pack2(Bm[i][j].v[0][2], Bm[i][j].v[0][3]);
          ba[i][j][2] = pack2(Bm[i][j].v[1][0], Bm[i][j].v[1][1]);
          ba[i][j][3] = pack2(Bm[i][j].v[1][2], Bm[i][j].v[1][3]);
          xa[i][j][0] = pack2(x[i][j].v[0][0], x[i][j].v[0][1]);
          xa[i][j][1] = pack2(x[i][j].v[0][2], x[i][j].v[0][3]);
          xa[i][j][2] = pack2(x[i][j].v[1][0], x[i][j].v[1][1]);
          xa[i][j][3] = pack2(x[i][j].v[1][2], x[i][j].v[1][3]);
        }
#pragma unroll
      for (int j = 0; j < NB; ++j) {
        uint32_t xb[NB][2][2];   // B fragments of Xb(kb, j): [kb][h][b0 / b1]
#pragma unroll
        for (int kb = 0; kb < NB; ++kb) {
          xb[kb][0][0] = movmatrix_trans(xa[kb][j][0]);
          xb[kb][0][1] = movmatrix_trans(xa[kb][j][1]);
          xb[kb][1][0] = movmatrix_trans(xa[kb][j][2]);
          xb[kb][1][1] = movmatrix_trans(xa[kb][j][3]);
        }
#pragma unroll
        for (int i = 0; i < NB; ++i)
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            x[i][j].v[h][0] *= s0[i];
            x[i][j].v[h][1] *= s0[i];
            x[i][j].v[h][2] *= s1[i];
            x[i][j].v[h][3] *= s1[i];
#pragma unroll
            for (int kb = 0; kb < NB; ++kb) mma_bf16(x[i][j].v[h], ba[i][kb], xb[kb][h][0], xb[kb][h][1]);
          }
      }
    }

    // ---------------- F: untile + scaled, weight-decayed write (Eq. 4.6) ---------------
    const float keep = 1.f - hp.lr * hp.wd;
    const float stepsz = step_mode ? -hp.lr * hp.scale_c * cur.tau_base : 1.f;
#pragma unroll
    for (int r = 0; r < kRowsPerLane; ++r) {
      const int i = r >> 1, rr = r & 1;
      uint32_t ww[kLaneBytes / 4], wo[kLaneBytes / 4];
      if (step_mode) read_row(cur, buf, 2, cur.pw, cur.sw, r, ww);
#pragma unroll
      for (int q = 0; q < kLaneBytes / 4; ++q) {
        float o0 = stepsz * x[i][q >> 1].v[q & 1][2 * rr], o1 = stepsz * x[i][q >> 1].v[q & 1][2 * rr + 1];
        if (step_mode) {
          o0 = fmaf(keep, bf_lo(ww[q]), o0);
          o1 = fmaf(keep, bf_hi(ww[q]), o1);
        }
        wo[q] = pack2(o0, o1);
      }
      write_row(cur, cur.pw, cur.sw, r, wo);
    }
    cur = nxt;
    buf ^= 1;
    it = nx;
  }
  cp_async_wait_all();
}

}  // namespace

cudaError_t launch_warp(const LaunchArgs& a, cudaStream_t s) {
  if (a.n_items < 1) return cudaSuccess;
  if (a.T != 16 && a.T != 32) return cudaErrorInvalidValue;
  const int per_sm = a.T == 16 ? Cfg<1>::kBlocksPerSm : Cfg<2>::kBlocksPerSm;
  const int warps = a.T == 16 ? Cfg<1>::kWarps : Cfg<2>::kWarps;
  const size_t smem = (size_t)warps * 2 * 3 * a.T * a.T * 2;
  cudaError_t e;
  if (a.T == 16) {
    static DeviceOnce once;
    e = configure_smem_once(once, himuon_warp_kernel<1>, (int)smem);
  } else {
    static DeviceOnce once;
    e = configure_smem_once(once, himuon_warp_kernel<2>, (int)smem);
  }
  if (e != cudaSuccess) return e;
  long long grid = (a.n_items + warps - 1) / warps;
  const long long cap = (long long)device_sm_count() * per_sm;
  if (grid > cap) grid = cap;
  if (a.T == 16) himuon_warp_kernel<1><<<(unsigned)grid, warps * 32, smem, s>>>(a.layers, a.items, a.n_items, a.mode, a.hp);
  else himuon_warp_kernel<2><<<(unsigned)grid, warps * 32, smem, s>>>(a.layers, a.items, a.n_items, a.mode, a.hp);
  return cudaGetLastError();
}

}  // namespace himuon
