// Tensor-core path of the HiMuon hot path for T = 64, bf16 storage (sm_100a: TMA + tcgen05 + TMEM).
//
// A tcgen05 MMA works on 128 TMEM lanes, so TWO 64 x 64 tiles of the work list (they may belong to
// different layers) are stacked into one 128 x 64 "super-tile" X' = [X_0; X_1] and every product of a
// Newton-Schulz step (Eq. 2.2) is one 128 x 128 x 64 MMA whose DIAGONAL 64 x 64 blocks
// are the per-tile products; the off-diagonal blocks mix the two tiles and are never read:
//   MMA1  ACC = X' X'^T            block (b, b) = X_b X_b^T = Ah_b
//   MMA2  ACC = Ot' Ot'^T          block (b, b) = Ot_b Ot_b^T      (Ot' = [Ot_0; Ot_1], 128 x 64)
//   MMA3  ACC = B' [X_0 | X_1]     block (b, b) = offdiag(B_b) X_b (B' = [B_0; B_1], 128 x 64; the
//                                  B operand is the stacked X' read MN-major, N = 2 x 64)
// Half of each MMA is wasted; the epilogues touch only the useful 64 accumulator columns of a row, so
// CUDA-core work per matrix element equals that of the T = 128 kernel.  Everything else (operands in
// TMEM, fp32 iterate in registers, fp32 diagonal of B as a row scaling, TMA prefetch, independent slots per
// CTA - three here, since a slot needs only 48 KB of shared memory, 160 TMEM columns and 32 state registers) follows kernels_tc128.cu, whose header states the per-tile algorithm and its citations.
//
// Thread (t, h) of a slot: row t of the super-tile (tile b = t >> 6, TMEM lane t), column half h of that
// tile (columns 32h..32h+31, i.e. accumulator columns 64b + 32h ..).
#include <cuda_bf16.h>
#include <stddef.h>

#include "himuon_internal.h"
#include "sm100_ptx.cuh"
#include "tc_common.cuh"

namespace himuon {
namespace {

using namespace ptx;
using namespace tc;

constexpr int T = 64;
constexpr int kPack = 2;                         // tiles per super-tile
constexpr int kSlots = 3;                        // independent super-tiles in flight per CTA (TMEM: 3 x 160 columns)
constexpr int kSlotThreads = 256;                // 8 warps: 4 lane quadrants x 2 column halves
constexpr int kThreads = kSlots * kSlotThreads;
constexpr uint32_t kTileBytes = T * T * 2;       // 8 KB: one bf16 tile = 64 rows x 128 B (one swizzle span wide)
constexpr uint32_t kBufBytes = kPack * kTileBytes;   // 16 KB: a stacked 128 x 64 operand
constexpr uint32_t kSlotBytes = 3 * kBufBytes;   // XB, OB, ST
constexpr uint32_t kCtrlBytes = 8192;
constexpr uint32_t kSmemBytes = kSlots * kSlotBytes + kCtrlBytes + 1024;  // + alignment slack
constexpr uint32_t kSlotCols = 160;              // TMEM columns per slot: ACC 128 (fp32) + OPA 32 (bf16 pairs)
constexpr uint32_t kOpaCol = 128;

struct SlotCtrl {
  unsigned long long mma_bar;   // tcgen05.commit of MMA1 / MMA2 / MMA3
  unsigned long long ld_bar;    // TMA loads of G (and M) of the next super-tile
  unsigned long long w_bar;     // TMA load of W
  float dpart[2][128];          // per column half: partial d_t = sum_j Xh_tj^2
  float spart[2][128];          // per column half: sum_j ACC_tj^2
  float red[8];
};
struct Ctrl {
  SlotCtrl slot[kSlots];
  uint32_t tmem_base;
};
static_assert(sizeof(Ctrl) <= kCtrlBytes, "control block too large");

// 16-byte chunk c (0..3) of this thread's 32 columns: rowaddr = buf + t*128 + (((4h) ^ (t&7)) << 4).
__device__ __forceinline__ uint32_t chunk_addr(uint32_t rowaddr, int c) { return rowaddr ^ ((uint32_t)c << 4); }

// K-major stacked operand (128 rows, K = 64 contiguous = one 128-byte swizzle span): k-step kk = 32 B.
__device__ __forceinline__ uint64_t desc_kmajor(uint32_t buf, int kk) {
  return make_smem_desc_sw128(buf + kk * 32, 16, 1024);
}
// The same buffer read MN-major: rows = K index within a tile (16 per k-step), N = 2 x 64 contiguous
// elements, the second 64 (tile 1) kTileBytes further (leading byte offset); 8-row groups 1024 B apart.
__device__ __forceinline__ uint64_t desc_mnmajor(uint32_t buf, int kk) {
  return make_smem_desc_sw128(buf + kk * 2048, kTileBytes, 1024);
}

__device__ __forceinline__ void issue_gram(uint32_t acc, uint32_t opa, uint32_t buf, uint32_t bar) {
  constexpr uint32_t idesc = make_idesc_bf16(128, 128, 0, 0);
#pragma unroll
  for (int kk = 0; kk < T / 16; ++kk) umma_bf16_ts(acc, opa + 8 * kk, desc_kmajor(buf, kk), idesc, kk ? 1u : 0u);
  umma_commit(bar);
}
__device__ __forceinline__ void issue_bx(uint32_t acc, uint32_t opa, uint32_t buf_x, uint32_t bar) {
  constexpr uint32_t idesc = make_idesc_bf16(128, 128, 0, 1);
#pragma unroll
  for (int kk = 0; kk < T / 16; ++kk) umma_bf16_ts(acc, opa + 8 * kk, desc_mnmajor(buf_x, kk), idesc, kk ? 1u : 0u);
  umma_commit(bar);
}

__global__ void __launch_bounds__(kThreads, 1)
himuon_tc64_kernel(const LayerDev* __restrict__ layers, const CUtensorMap* __restrict__ tmaps,
                   const WorkItem* __restrict__ items, long long n_items, int mode, himuon_hparams hp) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
  Ctrl* ctrl = reinterpret_cast<Ctrl*>(smem_raw + (smem0 - smem_u32(smem_raw)) + kSlots * kSlotBytes);

  const int tid = threadIdx.x;
  // warp-uniform in the compiler's eyes too (a shuffle result is uniform): what the MMA issue derives from it
  // (descriptors, TMEM and barrier addresses) then lives in uniform registers
  const int warp_id = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int slot = warp_id / (kSlotThreads / 32);
  const int ts = tid % kSlotThreads;
  const int w = warp_id % (kSlotThreads / 32);   // warp of the slot
  const int wq = w & 3;                // TMEM lane quadrant of this warp (= warp index in the CTA mod 4)
  const int h = w >> 2;                // column half of the thread's tile
  const int lane = tid & 31;
  const int t = wq * 32 + lane;        // row of the super-tile / TMEM lane
  const int b = t >> 6;                // which of the two stacked tiles
  const bool lead = (ts == 0);
  const bool step_mode = (mode == MODE_STEP);
  const bool own = ((wq & 1) == h);    // warp-uniform: this thread's 32 columns hold the diagonal element of row t
  const int dword = (lane & 15) >> 1;  // ... in 16-column chunk lane>>4, packed word dword, half lane&1
  const uint32_t dkeep = (lane & 1) ? 0x0000ffffu : 0xffff0000u;

  const uint32_t XB = smem0 + slot * kSlotBytes;
  const uint32_t OB = XB + kBufBytes;
  const uint32_t ST = OB + kBufBytes;
  const uint32_t rowoff = (uint32_t)t * 128u + ((((uint32_t)h << 2) ^ (uint32_t)(t & 7)) << 4);
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
  const uint32_t acc_t = tmem_slot + lane_off + 64u * b + 32u * h;       // this thread's 32 useful accumulator columns
  const uint32_t opa_t = tmem_slot + lane_off + kOpaCol + 16u * h;       // this thread's 16 packed operand columns
  const uint32_t ACCd = tmem_slot, OPAd = tmem_slot + kOpaCol;
  const uint32_t bar_id = 1 + slot;

  uint32_t ph_mma = 0, ph_ld = 0, ph_w = 0;
  auto wait_mma = [&]() {   // one warp polls, the others sleep on a hardware barrier
    if (w == 0) mbar_wait(mma_bar, ph_mma);
    named_bar_sync(8 + slot, kSlotThreads);
    ph_mma ^= 1;
    tc_fence_after_sync();
  };
  const float qs = sqrtf(sqrtf(hp.c));         // state Xh = c^(1/4) X, see kernels_tc128.cu
  const float beta_h = hp.b / sqrtf(hp.c);
  const long long n_super = (n_items + kPack - 1) / kPack;
  const long long stride = (long long)gridDim.x * kSlots;

  // tile j (0 / 1) of super-tile s; a missing second tile repeats the first one (its stores are skipped)
  auto item_at = [&](long long s, int j) {
    long long i = s * kPack + j;
    if (i >= n_items) i = s * kPack;
    WorkItem wi;
    if (items) wi = items[i];
    else { wi.layer = 0; wi.r = (int)i; wi.c = 0; wi.pad = 0; }
    return wi;
  };
  auto issue_g = [&](long long s) {      // G of both tiles -> OB; arms ld_bar for G and (step mode) M
    mbar_arrive_expect_tx(ld_bar, step_mode ? 2 * kBufBytes : kBufBytes);
#pragma unroll
    for (int j = 0; j < kPack; ++j) {
      const WorkItem wi = item_at(s, j);
      tma_load_2d(OB + j * kTileBytes, tmaps + 3 * wi.layer + 1, wi.c * T, wi.r * T, ld_bar);
    }
  };
  auto issue_m = [&](long long s) {      // M of both tiles -> XB
#pragma unroll
    for (int j = 0; j < kPack; ++j) {
      const WorkItem wi = item_at(s, j);
      tma_load_2d(XB + j * kTileBytes, tmaps + 3 * wi.layer + 2, wi.c * T, wi.r * T, ld_bar);
    }
  };

  long long it = (long long)blockIdx.x * kSlots + slot;
  if (lead && it < n_super) {
    issue_g(it);
    if (step_mode) issue_m(it);
  }

  for (; it < n_super; it += stride) {
    const WorkItem wi = item_at(it, b);                      // this thread's tile
    const float tau_base = layers[wi.layer].tau_base;
    const bool second_valid = it * kPack + 1 < n_items;
    const long long nxt = it + stride;
    bool g_issued = false, m_issued = false, w_issued = false;   // meaningful in the lead thread only

    auto issue_w = [&]() {               // W of both tiles -> ST (after M' has left it)
      tma_wait_group_read0();
      mbar_arrive_expect_tx(w_bar, kBufBytes);
#pragma unroll
      for (int j = 0; j < kPack; ++j) {
        const WorkItem wj = item_at(it, j);
        tma_load_2d(ST + j * kTileBytes, tmaps + 3 * wj.layer + 0, wj.c * T, wj.r * T, w_bar);
      }
      w_issued = true;
    };
    auto store_st = [&](int which) {     // ST -> M (which = 2) or W (which = 0) of both tiles
#pragma unroll
      for (int j = 0; j < kPack; ++j) {
        if (j == 1 && !second_valid) continue;
        const WorkItem wj = item_at(it, j);
        tma_store_2d(tmaps + 3 * wj.layer + which, wj.c * T, wj.r * T, ST + j * kTileBytes);
      }
      tma_commit_group();
    };

    // ---------------- P: momentum, normalise ---------------------------------------------------
    if (lead) {
      tma_wait_group_read0();   // the previous super-tile's stores out of ST have been read
      mbar_arrive(ld_bar);
    }
    mbar_wait(ld_bar, ph_ld);
    ph_ld ^= 1;

    f2 xs[16];                  // fp32 state: this thread's 32 columns of row t, as packed pairs
    f2 ss2 = pk2(0.f, 0.f);
    const f2 beta2 = pk2(hp.beta, hp.beta);
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const uint4 gv = lds128(chunk_addr(orow, c));
      const uint32_t gw[4] = {gv.x, gv.y, gv.z, gv.w};
      if (step_mode) {
        const uint4 mv = lds128(chunk_addr(xrow, c));
        const uint32_t mw[4] = {mv.x, mv.y, mv.z, mv.w};
        uint32_t mo[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const f2 g2 = pk2u(gw[e] << 16, gw[e] & 0xffff0000u);
          const f2 m2 = fma2(beta2, pk2u(mw[e] << 16, mw[e] & 0xffff0000u), g2);   // M' = beta M + G
          mo[e] = cvt_bf16x2(m2);
          const f2 h2 = hp.nesterov ? fma2(beta2, m2, g2) : m2;                    // Ghat
          ss2 = fma2(h2, h2, ss2);
          xs[4 * c + e] = h2;
        }
        sts128(chunk_addr(srow, c), make_uint4(mo[0], mo[1], mo[2], mo[3]));
      } else {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const f2 h2 = pk2u(gw[e] << 16, gw[e] & 0xffff0000u);
          ss2 = fma2(h2, h2, ss2);
          xs[4 * c + e] = h2;
        }
      }
    }
    float s0, s1;
    upk2(ss2, s0, s1);
    const float ss = s0 + s1;
    float tot = ss;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
    if (lane == 0) sc->red[w] = tot;
    fence_proxy_async_smem();          // M' in ST -> visible to the TMA store
    named_bar_sync(bar_id, kSlotThreads);
    if (lead && step_mode) store_st(2);
    // Frobenius norm of this thread's tile: its 64 rows are lane quadrants 2b and 2b+1, both column halves
    tot = (sc->red[2 * b] + sc->red[2 * b + 1]) + (sc->red[2 * b + 4] + sc->red[2 * b + 5]);
    const float nrm = sqrtf(tot);
    const float inv = nrm > 0.f ? qs / (nrm + hp.eps) : 0.f;   // Phi_K(0) = 0
    sc->dpart[h][t] = ss * inv * inv;                           // partial diag(Ah)_t in fp32
    {
      const f2 inv2 = pk2(inv, inv);
#pragma unroll
      for (int q = 0; q < 2; ++q) {
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
    if (w == 0 && hp.K > 0) {
      if (elect_one()) {
        tc_fence_after_sync();
        issue_gram(ACCd, OPAd, XB, mma_bar);
      }
      __syncwarp();
    }
    float di = sc->dpart[0][t] + sc->dpart[1][t];   // d_t = (Ah)_tt in fp32, from the fp32 state

    // ---------------- K Newton-Schulz steps ---------------------------------------------------
#pragma unroll 1
    for (int k = 0; k < hp.K; ++k) {
      const bool last = (k + 1 == hp.K);
      // ---- E1: block (b, b) of ACC = Ah_b
      wait_mma();
      {
        // Ot = offdiag(Ah) + diag(d + beta/2), rounded to bf16: for i != j
        //   (Ot Ot^T)_ij = (O^2)_ij + (beta + d_i + d_j) O_ij = (beta Ah + Ah^2)_ij = B_ij.
        const uint32_t dval = (pack_bf16(fmaf(0.5f, beta_h, di), 0.f) & 0xffffu) << ((lane & 1) * 16);
        f2 Sa = pk2(0.f, 0.f), Sb = Sa;
        uint32_t r[2][16];
        tmem_ld16(acc_t, r[0]);
        tmem_ld16(acc_t + 16, r[1]);
        tmem_wait_ld();
#pragma unroll
        for (int q = 0; q < 2; ++q) {
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const f2 o01 = pk2u(r[q][4 * j], r[q][4 * j + 1]), o23 = pk2u(r[q][4 * j + 2], r[q][4 * j + 3]);
            Sa = fma2(o01, o01, Sa);
            Sb = fma2(o23, o23, Sb);
          }
          uint32_t p[8];
          pack16(r[q], p);
          if (own) set_one(p, (lane >> 4) == q ? dword : 8, dkeep, dval);
          sts128(chunk_addr(orow, 2 * q), make_uint4(p[0], p[1], p[2], p[3]));
          sts128(chunk_addr(orow, 2 * q + 1), make_uint4(p[4], p[5], p[6], p[7]));
          tmem_st8(opa_t + 8 * q, p);
        }
        float s0, s1;
        upk2(add2(Sa, Sb), s0, s1);
        sc->spart[h][t] = s0 + s1;
      }
      if (lead && step_mode && !w_issued) issue_w();         // M' has left ST by now: fetch W into it
      tmem_wait_st();
      fence_proxy_async_smem();
      tc_fence_before_sync();
      named_bar_sync(bar_id, kSlotThreads);
      if (w == 0) {
        if (elect_one()) {
          tc_fence_after_sync();
          issue_gram(ACCd, OPAd, OB, mma_bar);
        }
        __syncwarp();
      }
      // a + B_tt, B_tt = beta d_t + (Ah^2)_tt
      const float si = hp.a + fmaf(beta_h, di, sc->spart[0][t] + sc->spart[1][t]);

      // ---- E2: block (b, b) of ACC = B_b off the diagonal
      wait_mma();
      if (lead && last && nxt < n_super) {                   // OB is free: fetch the next super-tile's G
        issue_g(nxt);
        g_issued = true;
      }
      {
        uint32_t r[2][16];
        tmem_ld16(acc_t, r[0]);
        tmem_ld16(acc_t + 16, r[1]);
        tmem_wait_ld();
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          uint32_t p[8];
          pack16(r[q], p);
          if (own) set_one(p, (lane >> 4) == q ? dword : 8, dkeep, 0u);
          tmem_st8(opa_t + 8 * q, p);
        }
      }
      tmem_wait_st();
      tc_fence_before_sync();
      named_bar_sync(bar_id, kSlotThreads);
      if (w == 0) {
        if (elect_one()) {
          tc_fence_after_sync();
          issue_bx(ACCd, OPAd, XB, mma_bar);
        }
        __syncwarp();
      }

      // ---- E3: Xh = (a + B_tt) Xh + offdiag(B) Xh
      wait_mma();
      if (lead && last && step_mode && g_issued) {           // XB is free: fetch the next super-tile's M
        issue_m(nxt);
        m_issued = true;
      }
      {
        const f2 si2 = pk2(si, si);
        f2 Da = pk2(0.f, 0.f), Db = Da;
        uint32_t r[2][16];
        tmem_ld16(acc_t, r[0]);
        tmem_ld16(acc_t + 16, r[1]);
        tmem_wait_ld();
#pragma unroll
        for (int q = 0; q < 2; ++q) {
#pragma unroll
          for (int j = 0; j < 8; ++j) xs[8 * q + j] = fma2(xs[8 * q + j], si2, pk2u(r[q][2 * j], r[q][2 * j + 1]));
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
        named_bar_sync(bar_id, kSlotThreads);
        if (w == 0) {
          if (elect_one()) {
            tc_fence_after_sync();
            issue_gram(ACCd, OPAd, XB, mma_bar);
          }
          __syncwarp();
        }
        di = sc->dpart[0][t] + sc->dpart[1][t];
      } else {
        tc_fence_before_sync();
      }
    }

    // ---------------- F: untile + scaled, weight-decayed write --------------------------------
    if (step_mode) {
      if (lead && !w_issued) issue_w();                      // K = 0: W was not prefetched
      mbar_wait(w_bar, ph_w);
      ph_w ^= 1;
    }
    {
      const float keep = 1.f - hp.lr * hp.wd;
      const float unq = 1.f / qs;                                   // undo the c^(1/4) state scaling
      const float stepsz = step_mode ? -hp.lr * hp.scale_c * tau_base * unq : unq;
      const f2 step2 = pk2(stepsz, stepsz), keep2 = pk2(keep, keep);
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t p[4];
        if (step_mode) {
          const uint4 wv = lds128(chunk_addr(srow, c));
          const uint32_t ww[4] = {wv.x, wv.y, wv.z, wv.w};
#pragma unroll
          for (int e = 0; e < 4; ++e)
            p[e] = cvt_bf16x2(fma2(keep2, pk2u(ww[e] << 16, ww[e] & 0xffff0000u), mul2(step2, xs[4 * c + e])));
        } else {
#pragma unroll
          for (int e = 0; e < 4; ++e) p[e] = cvt_bf16x2(mul2(step2, xs[4 * c + e]));
        }
        sts128(chunk_addr(srow, c), make_uint4(p[0], p[1], p[2], p[3]));
      }
    }
    fence_proxy_async_smem();
    named_bar_sync(bar_id, kSlotThreads);
    if (lead) {
      store_st(0);
      if (nxt < n_super) {                                   // whatever was not prefetched during the steps
        if (!g_issued) issue_g(nxt);
        if (step_mode && !m_issued) issue_m(nxt);
      }
    }
  }

  if (lead) tma_wait_group0();
  tc_fence_before_sync();
  __syncthreads();
  if (tid < 32) tmem_dealloc<512>(ctrl->tmem_base);
}

}  // namespace

cudaError_t launch_tc64(const LaunchArgs& a, cudaStream_t s) {
  static DeviceOnce once;   // per device, thread-safe
  cudaError_t e = configure_smem_once(once, himuon_tc64_kernel, (int)kSmemBytes);
  if (e != cudaSuccess) return e;
  const long long n_super = (a.n_items + kPack - 1) / kPack;
  long long grid = (n_super + kSlots - 1) / kSlots;
  const int sms = device_sm_count();
  if (grid > sms) grid = sms;
  if (grid < 1) return cudaSuccess;
  himuon_tc64_kernel<<<(unsigned)grid, kThreads, kSmemBytes, s>>>(a.layers, a.tmaps, a.items, a.n_items, a.mode, a.hp);
  return cudaGetLastError();
}

}  // namespace himuon
