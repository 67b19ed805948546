// Tensor-core path of the HiMuon hot path for T = 128, bf16 storage (sm_100a: TMA + tcgen05 + TMEM).
//
// One persistent CTA per SM holds TWO tiles in flight ("slots").  A slot is served by 8 warps:
// thread (t, h) owns row t of the tile (= TMEM lane t) and the column half h (columns 64h..64h+63).
// While one slot's warps run an epilogue on the CUDA cores, the other slot's MMAs run on the tensor
// pipe.  What the profile of the previous version showed (profiles/r1_tc128_v2_ncu_full.md) shaped
// this one: an SS-mode 128x128x16 MMA reads 8 KB of operands per 64 cycles, i.e. the whole
// shared-memory data path, and the epilogues' own smem traffic competes with it.  Here
//   * the A operand of every MMA lives in tensor memory (tcgen05.mma with A in TMEM), so an MMA
//     takes half the smem bandwidth and B_b (the A operand of MMA3) never touches smem;
//   * the fp32 iterate X lives in REGISTERS (64 per thread), which frees TMEM for the operand and
//     removes the separate "X <- (a + B_tt) X" pass over tensor memory;
//   * the next tile's G and M and this tile's W are fetched by TMA while the NS steps run.
//
// Per tile (Alg. 4.1; Eq. 2.2-2.3; Eq. 4.6), everything between the TMA loads of
// G, M, W and the TMA stores of M, W stays on chip:
//   P   G, M (smem) -> M' = beta M + G; Ghat = G + beta M' (Nesterov) | M'; M' -> TMA store;
//       Xh0 = q Ghat / (||Ghat||_F + eps), q = c^(1/4): fp32 in registers (state),
//       bf16 in smem XB (B operand) and in TMEM OPA (A operand)
//       (with the state scaled by q: Ah = Xh Xh^T = sqrt(c) A and B = bA + cA^2 = beta Ah + Ah^2,
//        beta = b / sqrt(c), so no accumulator ever needs a rescale by c)
//   K x MMA1  ACC  = Xb Xb^T                                   (Ah)
//       E1    Ot = bf16(offdiag(ACC) + diag(d + beta/2)) -> smem OB + TMEM OPA,  d_t = ||Xh row t||^2 (fp32);
//             S_t = sum_j ACC_tj^2 = (Ah^2)_tt  (fp32)
//       MMA2  ACC  = Ot Ot^T      (=> ACC_ij = (O^2)_ij + (beta + d_i + d_j) O_ij = B_ij for i != j)
//       E2    Bb = bf16(ACC), diagonal zeroed -> TMEM OPA
//       MMA3  ACC  = Bb Xb                                     (offdiag(B) Xh)
//       E3    X <- (a + B_tt) X + ACC, B_tt = beta d_t + S_t (fp32 row scaling, registers);
//             Xb = bf16(X) -> smem XB + TMEM OPA;  d_t = sum_j X_tj^2
//   F   W (smem, prefetched) ; W' = (1 - lr wd) W - lr tau X_K / q -> TMA store (Phi mode: X_K / q)
// The diagonals of A and B (O(1) numbers whose bf16 rounding would dominate the error) never pass
// through bf16: they act as fp32 row scalings.  DESIGN.md "Numerical scheme" derives the algebra.
//
// Ragged edge tiles: the TMA loads zero-fill outside H x W (= the zero padding of B_T,
// PAPER.md:51-53) and the TMA stores clip (= the crop of B_T^-1); padded rows and
// columns stay exactly zero through Eq. 2.2.
#include <cuda_bf16.h>
#include <stddef.h>

#include "himuon_internal.h"
#include "sm100_ptx.cuh"
#include "tc_common.cuh"

namespace himuon {

// Debug stages (1 / 2 = return the raw accumulator after MMA1 / MMA2 of the first step) exist only in the
// -DHIMUON_DEBUG_STAGES build (libhimuon_debug.so, used by the stage tests); the product library has neither the
// global, nor the export, nor the branches in the kernel.
#ifdef HIMUON_DEBUG_STAGES
int g_tc128_debug_stage = 0;
constexpr bool kDebugStages = true;
#else
constexpr bool kDebugStages = false;
#endif

#ifdef HIMUON_TRACE   // development aid (not built into libhimuon.so): clock stamps of the two lead threads of CTA 0
__device__ long long g_trace128[2][16384];
__device__ int g_tn128[2];
#define TR(id) do { if (lead && blockIdx.x == 0 && g_tn128[slot] < 16384) g_trace128[slot][g_tn128[slot]++] = ((long long)(id) << 48) | (clock64() & 0xffffffffffffLL); } while (0)
#else
#define TR(id) do { } while (0)
#endif

namespace {

using namespace ptx;
using namespace tc;

constexpr int T = 128;
constexpr int kSlots = 2;
constexpr int kSlotThreads = 256;                // 8 warps: 4 lane quadrants x 2 column halves
constexpr int kThreads = kSlots * kSlotThreads;
constexpr uint32_t kTileBytes = T * T * 2;       // 32 KB: one bf16 tile
constexpr uint32_t kHalfBytes = kTileBytes / 2;  // one 64-column block (128 rows x 128 B)
constexpr uint32_t kSlotBytes = 3 * kTileBytes;  // XB, OB, ST
constexpr uint32_t kCtrlBytes = 8192;
constexpr uint32_t kSmemBytes = kSlots * kSlotBytes + kCtrlBytes + 1024;  // + alignment slack
constexpr uint32_t kSlotCols = 256;              // TMEM columns per slot: ACC 128 (fp32) + OPA 64 (bf16 pairs)
constexpr uint32_t kOpaCol = 128;

struct SlotCtrl {
  unsigned long long mma_bar;   // tcgen05.commit of MMA1 / MMA2 / MMA3
  unsigned long long ld_bar;    // TMA loads of G (and M) of the next tile
  unsigned long long w_bar;     // TMA load of W
  float dpart[2][T];            // per column half: partial d_t = sum_j Xh_tj^2
  float spart[2][T];            // per column half: sum_j ACC_tj^2
  float red[8];
};
struct Ctrl {
  SlotCtrl slot[kSlots];
  uint32_t tmem_base;
};
static_assert(sizeof(Ctrl) <= kCtrlBytes, "control block too large");

// A [128 x 128] bf16 tile is stored as two 64-column blocks in the 128-byte-swizzled K-major layout
// (what TMA SWIZZLE_128B writes and what the UMMA descriptors below read).  `rowaddr` =
// block(h) + t*128 + ((t&7)<<4); 16-byte chunk c (0..7) of this thread's 64 columns is then one XOR away.
__device__ __forceinline__ uint32_t chunk_addr(uint32_t rowaddr, int c) { return rowaddr ^ ((uint32_t)c << 4); }

// K-major operand (rows = M or N index, K contiguous): k-step kk covers K elements 16kk..16kk+15.
__device__ __forceinline__ uint64_t desc_kmajor(uint32_t tile, int kk) {
  return make_smem_desc_sw128(tile + (kk >> 2) * kHalfBytes + (kk & 3) * 32, 16, 1024);
}
// MN-major operand (rows = K index, N contiguous): k-step kk covers rows 16kk..16kk+15;
// the two 64-column blocks are kHalfBytes apart (leading byte offset), 8-row groups 1024 B apart.
__device__ __forceinline__ uint64_t desc_mnmajor(uint32_t tile, int kk) {
  return make_smem_desc_sw128(tile + kk * 2048, kHalfBytes, 1024);
}

// ACC (+)= OPA * tile^T  (A = bf16 [128 x 128] in TMEM, B = K-major smem tile)
__device__ __forceinline__ void issue_gram(uint32_t acc, uint32_t opa, uint32_t tile, uint32_t accumulate, uint32_t bar) {
  constexpr uint32_t idesc = make_idesc_bf16(T, T, 0, 0);
#pragma unroll
  for (int kk = 0; kk < T / 16; ++kk)
    umma_bf16_ts(acc, opa + 8 * kk, desc_kmajor(tile, kk), idesc, (accumulate | (uint32_t)kk) ? 1u : 0u);
  umma_commit(bar);
}
// ACC = OPA * tile  (A = bf16 [128 x 128] in TMEM, B = the K-major tile read MN-major, i.e. not transposed)
__device__ __forceinline__ void issue_bx(uint32_t acc, uint32_t opa, uint32_t tile_x, uint32_t bar) {
  constexpr uint32_t idesc = make_idesc_bf16(T, T, 0, 1);
#pragma unroll
  for (int kk = 0; kk < T / 16; ++kk) umma_bf16_ts(acc, opa + 8 * kk, desc_mnmajor(tile_x, kk), idesc, kk ? 1u : 0u);
  umma_commit(bar);
}

__global__ void __launch_bounds__(kThreads, 1)
himuon_tc128_kernel(const LayerDev* __restrict__ layers, const CUtensorMap* __restrict__ tmaps,
                    const WorkItem* __restrict__ items, long long n_items, int mode, himuon_hparams hp, int dbg_arg) {
  const int dbg = kDebugStages ? dbg_arg : 0;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
  Ctrl* ctrl = reinterpret_cast<Ctrl*>(smem_raw + (smem0 - smem_u32(smem_raw)) + kSlots * kSlotBytes);

  const int tid = threadIdx.x;
  // warp-uniform in the compiler's eyes too (a shuffle result is uniform): everything the MMA issue derives from
  // it - descriptors, TMEM addresses, barrier addresses - then lives in uniform registers
  const int warp_id = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int slot = warp_id / (kSlotThreads / 32);
  const int ts = tid % kSlotThreads;
  const int w = warp_id % (kSlotThreads / 32);   // warp of the slot
  const int wq = w & 3;                // TMEM lane quadrant of this warp (= warp index in the CTA mod 4)
  const int h = w >> 2;                // column half
  const int lane = tid & 31;
  const int t = wq * 32 + lane;        // row of the tile / TMEM lane
  const bool lead = (ts == 0);
  const bool step_mode = (mode == MODE_STEP);

  const uint32_t XB = smem0 + slot * kSlotBytes;
  const uint32_t OB = XB + kTileBytes;
  const uint32_t ST = OB + kTileBytes;
  const uint32_t rowoff = (uint32_t)h * kHalfBytes + (uint32_t)t * 128u + ((uint32_t)(t & 7) << 4);
  const uint32_t xrow = XB + rowoff, orow = OB + rowoff, srow = ST + rowoff;
  SlotCtrl* sc = &ctrl->slot[slot];
  const uint32_t mma_bar = smem_u32(&sc->mma_bar);
  const uint32_t ld_bar = smem_u32(&sc->ld_bar);
  const uint32_t w_bar = smem_u32(&sc->w_bar);

  if (tid == 0) {
    for (int s = 0; s < kSlots; ++s) {
      mbar_init(smem_u32(&ctrl->slot[s].mma_bar), 1);
      mbar_init(smem_u32(&ctrl->slot[s].ld_bar), 2);   // arrive.expect_tx at issue + "staging is free" arrive
      mbar_init(smem_u32(&ctrl->slot[s].w_bar), 1);
    }
    fence_mbar_init();
  }
  if (tid < 32) tmem_alloc<512>(smem_u32(&ctrl->tmem_base));
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem_slot = ctrl->tmem_base + slot * kSlotCols;        // lane 0: MMA operand / destination addresses
  const uint32_t lane_off = (uint32_t)(wq * 32) << 16;
  const uint32_t acc_t = tmem_slot + lane_off + 64u * h;                 // this thread's 64 accumulator columns
  const uint32_t opa_t = tmem_slot + lane_off + kOpaCol + 32u * h;       // this thread's 32 packed operand columns
  const uint32_t ACCd = tmem_slot, OPAd = tmem_slot + kOpaCol;
  const uint32_t bar_id = 1 + slot;

  uint32_t ph_mma = 0, ph_ld = 0, ph_w = 0;
  // One warp of the slot polls the MMA barrier; the others sleep on a hardware barrier, so that waiting
  // warps do not take issue slots from the other slot's epilogue.
  auto wait_mma = [&]() {
    if (w == 0) mbar_wait(mma_bar, ph_mma);
    named_bar_sync(3 + slot, kSlotThreads);
  };
  // The state is Xh = c^(1/4) X: then Ah = Xh Xh^T = sqrt(c) A and B = bA + cA^2 = beta Ah + Ah^2 with
  // beta = b / sqrt(c), so the accumulator after MMA2 is B itself (no rescale in E2).
  const float qs = sqrtf(sqrtf(hp.c));
  const float beta_h = hp.b / sqrtf(hp.c);
  const long long stride = (long long)gridDim.x * kSlots;

  // ---- TMA issue helpers (lead thread of the slot only) ----------------------------------------------
  auto item_at = [&](long long i) {
    WorkItem wi;
    if (items) wi = items[i];
    else { wi.layer = 0; wi.r = (int)i; wi.c = 0; wi.pad = 0; }
    return wi;
  };
  auto issue_g = [&](long long i) {      // G of tile i -> OB; arms ld_bar for G and (step mode) M
    const WorkItem wi = item_at(i);
    const CUtensorMap* map_g = tmaps + 3 * wi.layer + 1;
    mbar_arrive_expect_tx(ld_bar, step_mode ? 2 * kTileBytes : kTileBytes);
    tma_load_2d(OB, map_g, wi.c * T, wi.r * T, ld_bar);
    tma_load_2d(OB + kHalfBytes, map_g, wi.c * T + 64, wi.r * T, ld_bar);
  };
  auto issue_m = [&](long long i) {      // M of tile i -> XB
    const WorkItem wi = item_at(i);
    const CUtensorMap* map_m = tmaps + 3 * wi.layer + 2;
    tma_load_2d(XB, map_m, wi.c * T, wi.r * T, ld_bar);
    tma_load_2d(XB + kHalfBytes, map_m, wi.c * T + 64, wi.r * T, ld_bar);
  };

  long long it = (long long)blockIdx.x * kSlots + slot;
  if (lead && it < n_items) {
    issue_g(it);
    if (step_mode) issue_m(it);
  }

  for (; it < n_items; it += stride) {
    const WorkItem wi = item_at(it);
    const float tau_base = layers[wi.layer].tau_base;
    const CUtensorMap* map_w = tmaps + 3 * wi.layer + 0;
    const CUtensorMap* map_m = tmaps + 3 * wi.layer + 2;
    const int x0 = wi.c * T, y0 = wi.r * T;
    const long long nxt = it + stride;
    bool g_issued = false, m_issued = false, w_issued = false;   // meaningful in the lead thread only
    // the diagonal element (t, t): 16-column chunk t>>4 of the row, packed word (t&15)>>1, half t&1
    const int dchunk = t >> 4, dword = (t & 15) >> 1;
    const uint32_t dkeep = (t & 1) ? 0x0000ffffu : 0xffff0000u;

    // ---------------- P: momentum, normalise ---------------------------------------------------
    TR(0);
    if (lead) {
      tma_wait_group_read0();   // the previous tile's stores out of ST have been read
      mbar_arrive(ld_bar);
    }
    mbar_wait(ld_bar, ph_ld);
    ph_ld ^= 1;
    TR(1);

    f2 xs[32];                  // fp32 state: this thread's 64 columns of row t, as packed pairs
    float ss = 0.f;             // sum of squares of this thread's part of Ghat
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      const uint4 gv = lds128(chunk_addr(orow, c));
      const uint32_t gw[4] = {gv.x, gv.y, gv.z, gv.w};
      if (step_mode) {
        const uint4 mv = lds128(chunk_addr(xrow, c));
        const uint32_t mw[4] = {mv.x, mv.y, mv.z, mv.w};
        uint32_t mo[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const float g0 = bf16_lo(gw[e]), g1 = bf16_hi(gw[e]);
          const float m0 = fmaf(hp.beta, bf16_lo(mw[e]), g0), m1 = fmaf(hp.beta, bf16_hi(mw[e]), g1);
          mo[e] = pack_bf16(m0, m1);
          const float h0 = hp.nesterov ? fmaf(hp.beta, m0, g0) : m0;
          const float h1 = hp.nesterov ? fmaf(hp.beta, m1, g1) : m1;
          ss = fmaf(h0, h0, ss);
          ss = fmaf(h1, h1, ss);
          xs[4 * c + e] = pk2(h0, h1);
        }
        sts128(chunk_addr(srow, c), make_uint4(mo[0], mo[1], mo[2], mo[3]));
      } else {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const float h0 = bf16_lo(gw[e]), h1 = bf16_hi(gw[e]);
          ss = fmaf(h0, h0, ss);
          ss = fmaf(h1, h1, ss);
          xs[4 * c + e] = pk2(h0, h1);
        }
      }
    }
    float tot = ss;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
    if (lane == 0) sc->red[w] = tot;
    fence_proxy_async_smem();          // M' in ST -> visible to the TMA store
    named_bar_sync(bar_id, kSlotThreads);
    TR(2);
    if (lead && step_mode) {
      tma_store_2d(map_m, x0, y0, ST);
      tma_store_2d(map_m, x0 + 64, y0, ST + kHalfBytes);
      tma_commit_group();
    }
    tot = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) tot += sc->red[i];
    const float nrm = sqrtf(tot);
    const float inv = nrm > 0.f ? qs / (nrm + hp.eps) : 0.f;   // Phi_K(0) = 0
    sc->dpart[h][t] = ss * inv * inv;                           // partial diag(Ah)_t in fp32
    {
      const f2 inv2 = pk2(inv, inv);
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        uint32_t p[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          xs[8 * q + j] = mul2(xs[8 * q + j], inv2);
          p[j] = cvt_bf16x2(xs[8 * q + j]);
        }
        sts128(chunk_addr(xrow, 2 * q), make_uint4(p[0], p[1], p[2], p[3]));
        sts128(chunk_addr(xrow, 2 * q + 1), make_uint4(p[4], p[5], p[6], p[7]));
        tmem_st8(opa_t + 8 * q, p);
      }
    }
    tmem_wait_st();
    fence_proxy_async_smem();
    tc_fence_before_sync();
    named_bar_sync(bar_id, kSlotThreads);
    TR(3);
    if (w == 0 && hp.K > 0) {
      if (elect_one()) {
        tc_fence_after_sync();
        issue_gram(ACCd, OPAd, XB, 0u, mma_bar);
      }
      __syncwarp();
    }
    TR(4);
    float di = sc->dpart[0][t] + sc->dpart[1][t];   // d_t = (Ah)_tt in fp32, from the fp32 state

    bool dumped = false;   // debug stages: xs holds a raw accumulator dump instead of X_K
    // ---------------- K Newton-Schulz steps ---------------------------------------------------
#pragma unroll 1
    for (int k = 0; k < hp.K; ++k) {
      const bool last = (k + 1 == hp.K);
      // ---- E1: ACC = Ah = Xh Xh^T just landed
      wait_mma();
      ph_mma ^= 1;
      tc_fence_after_sync();
      TR(10);
      if (dbg == 1) { dumped = true; break; }
      {
        // Ot = offdiag(Ah) + diag(d + beta/2), rounded to bf16: then for i != j
        //   (Ot Ot^T)_ij = (O^2)_ij + (beta + d_i + d_j) O_ij = (beta Ah + Ah^2)_ij = B_ij.
        const uint32_t dval = (pack_bf16(fmaf(0.5f, beta_h, di), 0.f) & 0xffffu) << ((t & 1) * 16);
        f2 Sa = pk2(0.f, 0.f), Sb = Sa;
        uint32_t r[2][16];
        tmem_ld16(acc_t, r[0]);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          tmem_wait_ld();
          if (q < 3) tmem_ld16(acc_t + 16 * (q + 1), r[(q + 1) & 1]);
          uint32_t(&c)[16] = r[q & 1];
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const f2 o01 = pk2u(c[4 * j], c[4 * j + 1]), o23 = pk2u(c[4 * j + 2], c[4 * j + 3]);
            Sa = fma2(o01, o01, Sa);
            Sb = fma2(o23, o23, Sb);
          }
          uint32_t p[8];
          pack16(c, p);
          // warp-uniform test: this chunk pair holds the diagonal of the warp's rows
          if ((((h << 2) + q) >> 1) == wq) set_one(p, dchunk == (h << 2) + q ? dword : 8, dkeep, dval);
          sts128(chunk_addr(orow, 2 * q), make_uint4(p[0], p[1], p[2], p[3]));
          sts128(chunk_addr(orow, 2 * q + 1), make_uint4(p[4], p[5], p[6], p[7]));
          tmem_st8(opa_t + 8 * q, p);
        }
        float s0, s1;
        upk2(add2(Sa, Sb), s0, s1);
        sc->spart[h][t] = s0 + s1;
      }
      if (lead && step_mode && !w_issued) {                 // M' has left ST by now: fetch W into it
        tma_wait_group_read0();
        mbar_arrive_expect_tx(w_bar, kTileBytes);
        tma_load_2d(ST, map_w, x0, y0, w_bar);
        tma_load_2d(ST + kHalfBytes, map_w, x0 + 64, y0, w_bar);
        w_issued = true;
      }
      tmem_wait_st();
      fence_proxy_async_smem();
      tc_fence_before_sync();
      TR(11);
      named_bar_sync(bar_id, kSlotThreads);
      TR(12);
      if (w == 0) {
        if (elect_one()) {
          tc_fence_after_sync();
          issue_gram(ACCd, OPAd, OB, 0u, mma_bar);
        }
        __syncwarp();
      }
      TR(13);
      // a + B_tt, B_tt = beta d_t + (Ah^2)_tt
      const float si = hp.a + fmaf(beta_h, di, sc->spart[0][t] + sc->spart[1][t]);

      // ---- E2: ACC = B (off-diagonal)
      wait_mma();
      ph_mma ^= 1;
      tc_fence_after_sync();
      TR(20);
      if (dbg == 2) { dumped = true; break; }
      if (lead && last && nxt < n_items) {                  // OB is free: fetch the next tile's G
        issue_g(nxt);
        g_issued = true;
      }
      {
        uint32_t r[2][16];
        tmem_ld16(acc_t, r[0]);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          tmem_wait_ld();
          if (q < 3) tmem_ld16(acc_t + 16 * (q + 1), r[(q + 1) & 1]);
          uint32_t(&c)[16] = r[q & 1];
          uint32_t p[8];
          pack16(c, p);
          if ((((h << 2) + q) >> 1) == wq) set_one(p, dchunk == (h << 2) + q ? dword : 8, dkeep, 0u);
          tmem_st8(opa_t + 8 * q, p);
        }
      }
      tmem_wait_st();
      tc_fence_before_sync();
      TR(21);
      named_bar_sync(bar_id, kSlotThreads);
      TR(22);
      if (w == 0) {
        if (elect_one()) {
          tc_fence_after_sync();
          issue_bx(ACCd, OPAd, XB, mma_bar);
        }
        __syncwarp();
      }
      TR(23);

      // ---- E3: Xh = (a + B_tt) Xh + offdiag(B) Xh
      wait_mma();
      ph_mma ^= 1;
      tc_fence_after_sync();
      TR(30);
      if (lead && last && step_mode && g_issued) {          // XB is free: fetch the next tile's M
        issue_m(nxt);
        m_issued = true;
      }
      {
        const f2 si2 = pk2(si, si);
        f2 Da = pk2(0.f, 0.f), Db = Da;
        uint32_t r[2][16];
        tmem_ld16(acc_t, r[0]);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          tmem_wait_ld();
          if (q < 3) tmem_ld16(acc_t + 16 * (q + 1), r[(q + 1) & 1]);
          uint32_t(&c)[16] = r[q & 1];
#pragma unroll
          for (int j = 0; j < 8; ++j) xs[8 * q + j] = fma2(xs[8 * q + j], si2, pk2u(c[2 * j], c[2 * j + 1]));
          if (!last) {
            uint32_t p[8];
#pragma unroll
            for (int j = 0; j < 8; j += 2) {
              Da = fma2(xs[8 * q + j], xs[8 * q + j], Da);
              Db = fma2(xs[8 * q + j + 1], xs[8 * q + j + 1], Db);
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) p[j] = cvt_bf16x2(xs[8 * q + j]);
            sts128(chunk_addr(xrow, 2 * q), make_uint4(p[0], p[1], p[2], p[3]));
            sts128(chunk_addr(xrow, 2 * q + 1), make_uint4(p[4], p[5], p[6], p[7]));
            tmem_st8(opa_t + 8 * q, p);
          }
        }
        if (!last) {
          float d0, d1;
          upk2(add2(Da, Db), d0, d1);
          sc->dpart[h][t] = d0 + d1;
        }
      }
      if (!last) {
        tmem_wait_st();
        fence_proxy_async_smem();
        tc_fence_before_sync();
        TR(31);
        named_bar_sync(bar_id, kSlotThreads);
        TR(32);
        if (w == 0) {
          if (elect_one()) {
            tc_fence_after_sync();
            issue_gram(ACCd, OPAd, XB, 0u, mma_bar);
          }
          __syncwarp();
        }
        TR(33);
        di = sc->dpart[0][t] + sc->dpart[1][t];
      }
    }
    if (dumped) {   // tests only: return the raw accumulator instead of X_K
      uint32_t r[16];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        tmem_ld16(acc_t + 16 * q, r);
        tmem_wait_ld();
#pragma unroll
        for (int j = 0; j < 8; ++j) xs[8 * q + j] = pk2u(r[2 * j], r[2 * j + 1]);
      }
      tc_fence_before_sync();
    }

    // ---------------- F: untile + scaled, weight-decayed write --------------------------------
    TR(40);
    if (step_mode) {
      if (lead && !w_issued) {                               // K = 0 or a debug stage: W was not prefetched
        tma_wait_group_read0();
        mbar_arrive_expect_tx(w_bar, kTileBytes);
        tma_load_2d(ST, map_w, x0, y0, w_bar);
        tma_load_2d(ST + kHalfBytes, map_w, x0 + 64, y0, w_bar);
      }
      mbar_wait(w_bar, ph_w);
      ph_w ^= 1;
    }
    TR(41);
    {
      const float keep = 1.f - hp.lr * hp.wd;
      const float unq = dbg ? 1.f : 1.f / qs;                       // undo the c^(1/4) state scaling
      const float stepsz = step_mode ? -hp.lr * hp.scale_c * tau_base * unq : unq;
      const f2 step2 = pk2(stepsz, stepsz), keep2 = pk2(keep, keep);
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        uint32_t p[4];
        if (step_mode) {
          const uint4 wv = lds128(chunk_addr(srow, c));
          const uint32_t ww[4] = {wv.x, wv.y, wv.z, wv.w};
#pragma unroll
          for (int e = 0; e < 4; ++e)
            p[e] = cvt_bf16x2(fma2(keep2, pk2(bf16_lo(ww[e]), bf16_hi(ww[e])), mul2(step2, xs[4 * c + e])));
        } else {
#pragma unroll
          for (int e = 0; e < 4; ++e) p[e] = cvt_bf16x2(mul2(step2, xs[4 * c + e]));
        }
        sts128(chunk_addr(srow, c), make_uint4(p[0], p[1], p[2], p[3]));
      }
    }
    fence_proxy_async_smem();
    TR(42);
    named_bar_sync(bar_id, kSlotThreads);
    TR(43);
    if (lead) {
      tma_store_2d(map_w, x0, y0, ST);
      tma_store_2d(map_w, x0 + 64, y0, ST + kHalfBytes);
      tma_commit_group();
      if (nxt < n_items) {                                   // whatever was not prefetched during the steps
        if (!g_issued) issue_g(nxt);
        if (step_mode && !m_issued) issue_m(nxt);
      }
    }
    TR(44);
  }

  if (lead) tma_wait_group0();
  tc_fence_before_sync();
  __syncthreads();
  if (tid < 32) tmem_dealloc<512>(ctrl->tmem_base);
}

}  // namespace

cudaError_t launch_tc128(const LaunchArgs& a, cudaStream_t s) {
  static DeviceOnce once;   // per device, thread-safe
  cudaError_t e = configure_smem_once(once, himuon_tc128_kernel, (int)kSmemBytes);
  if (e != cudaSuccess) return e;
  long long grid = (a.n_items + kSlots - 1) / kSlots;
  const int sms = device_sm_count();
  if (grid > sms) grid = sms;
  if (grid < 1) return cudaSuccess;
#ifdef HIMUON_DEBUG_STAGES
  const int stage = g_tc128_debug_stage;
#else
  const int stage = 0;
#endif
  himuon_tc128_kernel<<<(unsigned)grid, kThreads, kSmemBytes, s>>>(a.layers, a.tmaps, a.items, a.n_items, a.mode, a.hp,
                                                                   stage);
  return cudaGetLastError();
}

}  // namespace himuon

#ifdef HIMUON_DEBUG_STAGES
extern "C" void himuon_debug_set_tc128_stage(int stage) { himuon::g_tc128_debug_stage = stage; }
#endif
#ifdef HIMUON_TRACE
extern "C" int himuon_debug_read_trace128(long long* out, int* n) {
  cudaMemcpyFromSymbol(n, himuon::g_tn128, sizeof(int) * 2, 0, cudaMemcpyDeviceToHost);
  return (int)cudaMemcpyFromSymbol(out, himuon::g_trace128, sizeof(long long) * 2 * 16384, 0, cudaMemcpyDeviceToHost);
}
extern "C" int himuon_debug_reset_trace128() {
  int z[2] = {0, 0};
  return (int)cudaMemcpyToSymbol(himuon::g_tn128, z, sizeof(z));
}
#endif
