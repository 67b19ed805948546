// Tensor-core path of the HiMuon hot path for T = 128, bf16 storage (sm_100a: TMA + tcgen05 + TMEM), with bf16 or
// - opt-in, HIMUON_PATH_FP8 - e4m3 operands in the three products of a Newton-Schulz step (one template).
//
// One persistent CTA per SM holds TWO tiles in flight ("slots").  Warp-specialised (round 2; what the clock-stamp
// traces of the round-1 kernel showed is in DESIGN.md section 7):
//   warps 0-7 / 8-15   epilogue warps of slot 0 / 1: thread (t, h) owns row t of the tile (= TMEM lane t) and the
//                      16-column chunks 2q + h, q = 0..3 (columns 32q + 16h .. + 15).  Interleaving the chunks puts
//                      the diagonal element of every row into iteration q = t >> 5 of BOTH column halves' warps, so
//                      every warp patches one chunk per phase (not two or none).  Straight-line code: these warps
//                      issue no MMA and no TMA, they only wait on and arrive at mbarriers.
//   warp 16            MMA issuer for both slots: waits for a slot's "operands written" mbarrier (256 arrivals),
//                      issues the 8 (bf16) / 4 (e4m3) tcgen05.mma of the next product from uniform registers and
//                      commits to the slot's "accumulator ready" mbarrier.  tcgen05.mma issue blocks while the tensor
//                      pipe's queue is full; in this warp that costs nothing.  The two slots are served first come,
//                      first served, so their products never interleave instruction by instruction.
//   warps 17 / 18      TMA producer of slot 0 / 1: loads G, M, W of the next tile as soon as the issuer's commits say
//                      a buffer is free, stores M' and W' when the epilogue warps say they are written.
//   (warp 19 idles: setmaxnreg moves registers by warpgroup.)  Control warps run at 24 registers, epilogue warps
//   at 112 (setmaxnreg).  The pool setmaxnreg redistributes is what the CTA was LAUNCHED with - 640 threads x 96
//   registers (the most a 640-thread block can get) = 60 K, not the SM's 64 K: 16 x 32 x 112 + 4 x 32 x 24 = 60 K
//   (asking for 120 deadlocks: measured).
// While one slot's warps run an epilogue on the CUDA cores, the other slot's product runs on the tensor pipe.
//   * the A operand of every MMA lives in tensor memory (tcgen05.mma with A in TMEM): an MMA takes half the smem
//     bandwidth of the SS form and B_b (the A operand of MMA3) never touches smem;
//   * the fp32 iterate X lives in REGISTERS (64 per thread).
//
// Buffers of a slot (32 KB each, 128-byte-swizzled K-major [128 x 64]-column blocks as TMA writes them):
//   OB   G (TMA) -> Xb = bf16(Xh), the B operand of MMA1 (K-major) and MMA3 (read MN-major), rewritten by E3
//   XB   M (TMA) -> M' in place -> TMA store;  then Ot, the B operand of MMA2, rewritten by E1
//   ST   W (TMA) -> W' in place -> TMA store   (Phi mode: the output tile)
// (e4m3: the operands use the first 16 KB of OB / XB as one [128 rows x 128 B] block.)
//
// Per tile (Alg. 4.1; Eq. 2.2-2.3; Eq. 4.6), everything between the TMA loads of G, M, W and the
// TMA stores of M', W' stays on chip:
//   P   M' = beta M + G; Ghat = G + beta M' (Nesterov) | M';  Xh0 = q Ghat / (||Ghat||_F + eps), q = c^(1/4):
//       fp32 in registers (state), bf16 in smem (B operand) and in TMEM OPA (A operand)
//       (with the state scaled by q: Ah = Xh Xh^T = sqrt(c) A and B = bA + cA^2 = beta Ah + Ah^2,
//        beta = b / sqrt(c), so no accumulator ever needs a rescale by c)
//   K x MMA1  ACC  = Xb Xb^T                                   (Ah)
//       E1    Ot = bf16(offdiag(ACC) + diag(d + beta/2)) -> smem XB + TMEM OPA,  d_t = ||Xh row t||^2 (fp32);
//             S_t = sum_j ACC_tj^2 = (Ah^2)_tt  (fp32)
//       MMA2  ACC  = Ot Ot^T      (=> ACC_ij = (O^2)_ij + (beta + d_i + d_j) O_ij = B_ij for i != j)
//       E2    Bb = bf16(ACC), diagonal zeroed -> TMEM OPA
//       MMA3  ACC  = Bb Xb                                     (offdiag(B) Xh)
//       E3    X <- (a + B_tt) X + ACC, B_tt = beta d_t + S_t (fp32 row scaling, registers);
//             Xb = bf16(X) -> smem OB + TMEM OPA;  d_t = sum_j X_tj^2
//   F   W' = (1 - lr wd) W - lr tau X_K / q -> TMA store (Phi mode: X_K / q)
// The diagonals of A and B (O(1) numbers whose bf16 rounding would dominate the error) never pass through bf16:
// they act as fp32 row scalings.  DESIGN.md "Numerical scheme" derives the algebra.
//
// e4m3 operands (F8 = true; PAPER.md:410-424 section 6.5, :440 "fp8e4m3 with per-tile dynamic
// scaling"): tcgen05.mma kind::f8f6f4, K = 32 per instruction.  Every tile is normalised by its own Frobenius norm
// before the first product (that IS the per-tile dynamic scale, Eq. 2.2), after which the operands are bounded a
// priori: |Xh_ij| <= ||Xh||_2 <= 1.2 c^(1/4) = 1.43, |Ah_ij| <= 2.05, |B_ij| <= 2.8.  Fixed power-of-two scales
// s_X = 256, s_O = 128, s_B = 128 therefore cannot saturate (e4m3 max 448) and keep typical entries in the normal
// range.  The accumulators come out scaled by s_X^2, s_O^2, s_B s_X and are unscaled in the epilogues.  Accumulation,
// the iterate, the diagonals, momentum and update stay fp32.  DESIGN.md section 5: accuracy (~0.1 per tile) and the
// failure mode on heavy-tailed tiles.
//
// Ragged edge tiles: the TMA loads zero-fill outside H x W (= the zero padding of B_T) and the TMA
// stores clip (= the crop of B_T^-1); padded rows and columns stay exactly zero through Eq. 2.2
// (PAPER.md:243).
#include <cuda_bf16.h>
#include <stddef.h>

#include "himuon_internal.h"
#include "sm100_ptx.cuh"
#include "tc_common.cuh"

namespace himuon {

// Debug stages (1 / 2 = return the raw accumulator after MMA1 / MMA2 of the first step) exist only in the
// -DHIMUON_DEBUG_STAGES build (libhimuon_debug.so, used by the stage tests); the product library has neither the
// globals, nor the exports, nor the branches in the kernel.
#ifdef HIMUON_DEBUG_STAGES
int g_tc128_debug_stage = 0;
int g_tc128_fp8_debug_stage = 0;
constexpr bool kDebugStages = true;
#else
constexpr bool kDebugStages = false;
#endif

#ifdef HIMUON_TRACE   // development aid (not built into libhimuon.so): clock stamps of CTA 0
__device__ long long g_trace128[4][16384];   // 0, 1: lead epilogue thread of slot 0 / 1; 2: issuer; 3: producer of slot 0
__device__ int g_tn128[4];
#define TRW(who, id) do { if (blockIdx.x == 0 && g_tn128[who] < 16384) g_trace128[who][g_tn128[who]++] = ((long long)(id) << 48) | (clock64() & 0xffffffffffffLL); } while (0)
#define TR(id) do { if (ts == 0) TRW(slot, id); } while (0)
#else
#define TRW(who, id) do { } while (0)
#define TR(id) do { } while (0)
#endif

namespace {

using namespace ptx;
using namespace tc;

constexpr int T = 128;
constexpr int kSlots = 2;
constexpr int kSlotThreads = 256;                // 8 warps: 4 lane quadrants x 2 column halves
constexpr int kEpiThreads = kSlots * kSlotThreads;
constexpr int kThreads = kEpiThreads + 128;      // + one control warpgroup: issuer, two producers, one idle warp
constexpr int kIssuerWarp = kEpiThreads / 32;
constexpr uint32_t kTileBytes = T * T * 2;       // 32 KB: one bf16 tile
constexpr uint32_t kHalfBytes = kTileBytes / 2;  // one 64-column block (128 rows x 128 B)
constexpr uint32_t kOp8Bytes = T * T;            // 16 KB: one e4m3 operand tile (128 rows x 128 B, one swizzle span)
constexpr uint32_t kSlotBytes = 3 * kTileBytes;  // XB, OB, ST
constexpr uint32_t kXB = 0, kOB = kTileBytes, kST = 2 * kTileBytes;
constexpr uint32_t kCtrlBytes = 8192;
constexpr uint32_t kSmemBytes = kSlots * kSlotBytes + kCtrlBytes + 1024;  // + alignment slack
constexpr uint32_t kSlotCols = 256;              // TMEM columns per slot: ACC 128 (fp32) + OPA 64 (bf16 pairs) / 32 (e4m3 quads)
constexpr uint32_t kOpaCol = 128;
constexpr float kSX = 256.f, kSO = 128.f, kSB = 128.f;   // e4m3 operand scales (powers of two)

struct SlotCtrl {
  unsigned long long opnd_full;   // epilogue -> issuer: operands of the next product are written (256 arrivals)
  unsigned long long mma_done;    // issuer (tcgen05.commit) -> epilogue: the accumulator is ready
  unsigned long long xb_mma_free; // issuer (commit after the tile's last MMA2) -> producer: XB may receive the next M
  unsigned long long ob_mma_free; // issuer (commit after the tile's last MMA3) -> producer: OB may receive the next G
  unsigned long long ld_full;     // producer (TMA) -> epilogue: G (and M) of the tile have landed
  unsigned long long w_full;      // producer (TMA) -> epilogue: W has landed in ST (Phi mode: ST is free)
  unsigned long long mp_full;     // epilogue -> producer: M' is written in XB (256 arrivals)
  unsigned long long xb_free;     // producer -> epilogue: the M' store has left XB, Ot may be written into it
  unsigned long long out_full;    // epilogue -> producer: W' (Phi mode: the output tile) is written in ST (256 arrivals)
  float tau[2];                   // tau_base of the tile, by tile parity (written by the producer before the loads)
  float dpart[2][T];              // per column half: partial d_t = sum_j Xh_tj^2
  float spart[2][T];              // per column half: sum_j ACC_tj^2
  float red[8];
};
struct Ctrl {
  SlotCtrl slot[kSlots];
  uint32_t tmem_base;
};
static_assert(sizeof(Ctrl) <= kCtrlBytes, "control block too large");

template <bool F8>
struct Fmt {
  static constexpr int kMmas = F8 ? T / 32 : T / 16;        // tcgen05.mma per product
  static constexpr int kWords = F8 ? 4 : 8;                 // packed 32-bit words per 16 columns
};

// K-major operand (rows = M or N index, K contiguous), k-step kk.
template <bool F8>
__device__ __forceinline__ uint64_t desc_kmajor(uint32_t tile, int kk) {
  if constexpr (F8) return make_smem_desc_sw128(tile + kk * 32, 16, 1024);                               // 32 elements = 32 B
  else return make_smem_desc_sw128(tile + (kk >> 2) * kHalfBytes + (kk & 3) * 32, 16, 1024);            // 16 elements = 32 B
}
// MN-major operand (rows = K index, N contiguous), k-step kk.
template <bool F8>
__device__ __forceinline__ uint64_t desc_mnmajor(uint32_t tile, int kk) {
  if constexpr (F8) return make_smem_desc_sw128(tile + kk * 4096, kOp8Bytes, 1024);     // 32 rows of 128 B
  else return make_smem_desc_sw128(tile + kk * 2048, kHalfBytes, 1024);                 // 16 rows; the two 64-column blocks kHalfBytes apart
}
template <bool F8>
__device__ __forceinline__ void umma_ts(uint32_t d, uint32_t a, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
  if constexpr (F8) umma_f8_ts(d, a, bdesc, idesc, acc);
  else umma_bf16_ts(d, a, bdesc, idesc, acc);
}
// ACC = OPA * tile^T (mn = false: Gram form, B K-major) or OPA * tile (mn = true: B read MN-major)
template <bool F8>
__device__ __forceinline__ void issue_product(uint32_t acc, uint32_t opa, uint32_t tile, bool mn) {
  const uint32_t id_k = F8 ? make_idesc_e4m3(T, T, 0, 0) : make_idesc_bf16(T, T, 0, 0);
  const uint32_t id_mn = F8 ? make_idesc_e4m3(T, T, 0, 1) : make_idesc_bf16(T, T, 0, 1);
  if (!mn) {
#pragma unroll
    for (int kk = 0; kk < Fmt<F8>::kMmas; ++kk) umma_ts<F8>(acc, opa + 8 * kk, desc_kmajor<F8>(tile, kk), id_k, kk ? 1u : 0u);
  } else {
#pragma unroll
    for (int kk = 0; kk < Fmt<F8>::kMmas; ++kk) umma_ts<F8>(acc, opa + 8 * kk, desc_mnmajor<F8>(tile, kk), id_mn, kk ? 1u : 0u);
  }
}

__device__ __forceinline__ void setmaxnreg_inc112() { asm volatile("setmaxnreg.inc.sync.aligned.u32 112;"); }
__device__ __forceinline__ void setmaxnreg_dec24() { asm volatile("setmaxnreg.dec.sync.aligned.u32 24;"); }

template <bool F8>
__global__ void __launch_bounds__(kThreads, 1)
himuon_tc128_kernel(const LayerDev* __restrict__ layers, const CUtensorMap* __restrict__ tmaps,
                    const WorkItem* __restrict__ items, long long n_items, int mode, himuon_hparams hp, int dbg_arg) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
  Ctrl* ctrl = reinterpret_cast<Ctrl*>(smem_raw + (smem0 - smem_u32(smem_raw)) + kSlots * kSlotBytes);
  const int dbg = kDebugStages ? dbg_arg : 0;

  const int tid = threadIdx.x;
  // warp-uniform for the compiler too (a shuffle result is uniform): what the control warps derive from it
  // (descriptors, TMEM and barrier addresses) lives in uniform registers
  const int warp_id = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const bool step_mode = (mode == MODE_STEP);

  if (tid == 0) {
    for (int s = 0; s < kSlots; ++s) {
      SlotCtrl* c = &ctrl->slot[s];
      mbar_init(smem_u32(&c->opnd_full), kSlotThreads);
      mbar_init(smem_u32(&c->mma_done), 1);
      mbar_init(smem_u32(&c->xb_mma_free), 1);
      mbar_init(smem_u32(&c->ob_mma_free), 1);
      mbar_init(smem_u32(&c->ld_full), 1);
      mbar_init(smem_u32(&c->w_full), 1);
      mbar_init(smem_u32(&c->mp_full), kSlotThreads);
      mbar_init(smem_u32(&c->xb_free), 1);
      mbar_init(smem_u32(&c->out_full), kSlotThreads);
    }
    fence_mbar_init();
  }
  if (warp_id == kIssuerWarp) tmem_alloc<512>(smem_u32(&ctrl->tmem_base));
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem_base = ctrl->tmem_base;

  const long long stride = (long long)gridDim.x * kSlots;
  // products per tile: 3 per Newton-Schulz step (debug stages stop after the first / second product of step 0)
  const int n_phases = dbg ? dbg : 3 * hp.K;

  if (warp_id >= kIssuerWarp) {
    setmaxnreg_dec24();
    if (warp_id == kIssuerWarp) {
      // ================= MMA issuer (one thread, both slots) =================================================
      if (elect_one()) {
        long long left[kSlots];
        int phase[kSlots] = {0, 0};
        uint32_t par[kSlots] = {0, 0};
#pragma unroll
        for (int s = 0; s < kSlots; ++s) {
          const long long g = (long long)blockIdx.x * kSlots + s;
          left[s] = n_items > g ? (n_items - g + stride - 1) / stride : 0;
        }
        while (left[0] > 0 || left[1] > 0) {
          bool any = false;
#pragma unroll
          for (int s = 0; s < kSlots; ++s) {
            SlotCtrl* c = &ctrl->slot[s];
            if (left[s] > 0 && mbar_test_wait(smem_u32(&c->opnd_full), par[s])) {
              any = true;
              par[s] ^= 1;
              tc_fence_after_sync();
              const uint32_t sb = smem0 + s * kSlotBytes;
              const uint32_t acc = tmem_base + s * kSlotCols, opa = acc + kOpaCol;
              if (n_phases == 0) {                     // K = 0: nothing to issue; P has consumed G and M
                umma_commit(smem_u32(&c->xb_mma_free));
                umma_commit(smem_u32(&c->ob_mma_free));
                --left[s];
              } else {
                const int which = phase[s] % 3;        // 0: Xb Xb^T (OB), 1: Ot Ot^T (XB), 2: Bb Xb (OB, MN-major)
                if (which == 0) issue_product<F8>(acc, opa, sb + kOB, false);
                else if (which == 1) issue_product<F8>(acc, opa, sb + kXB, false);
                else issue_product<F8>(acc, opa, sb + kOB, true);
                umma_commit(smem_u32(&c->mma_done));
                TRW(2, 100 + 10 * s + which);
                // XB holds Ot, read by MMA2 only: free after the tile's last MMA2 (debug stages: after the last product)
                if (phase[s] == (dbg ? n_phases - 1 : n_phases - 2)) umma_commit(smem_u32(&c->xb_mma_free));
                if (++phase[s] == n_phases) {
                  umma_commit(smem_u32(&c->ob_mma_free));
                  phase[s] = 0;
                  --left[s];
                }
              }
            }
          }
          (void)any;   // (no back-off: nanosleep(32) was measured - see DESIGN.md section 7)
        }
      }
      __syncwarp();
    } else if (warp_id <= kIssuerWarp + kSlots) {
      // ================= TMA producer of one slot (one thread) ===============================================
      const int slot = warp_id - kIssuerWarp - 1;
      if (elect_one()) {
        SlotCtrl* c = &ctrl->slot[slot];
        const uint32_t sb = smem0 + slot * kSlotBytes;
        const uint32_t XB = sb + kXB, OB = sb + kOB, ST = sb + kST;
        const uint32_t ld_full = smem_u32(&c->ld_full), w_full = smem_u32(&c->w_full);
        auto item_at = [&](long long i) {
          WorkItem wi;
          if (items) wi = items[i];
          else { wi.layer = 0; wi.r = (int)i; wi.c = 0; wi.pad = 0; }
          return wi;
        };
        auto load2 = [&](uint32_t dst, const CUtensorMap* map, const WorkItem& wi, uint32_t bar) {
          tma_load_2d(dst, map, wi.c * T, wi.r * T, bar);
          tma_load_2d(dst + kHalfBytes, map, wi.c * T + 64, wi.r * T, bar);
        };
        auto store2 = [&](const CUtensorMap* map, const WorkItem& wi, uint32_t src) {
          tma_store_2d(map, wi.c * T, wi.r * T, src);
          tma_store_2d(map, wi.c * T + 64, wi.r * T, src + kHalfBytes);
          tma_commit_group();
        };
        uint32_t p_mp = 0, p_xm = 0, p_om = 0, p_out = 0;
        long long it = (long long)blockIdx.x * kSlots + slot;
        int n = 0;                                     // tile counter of this slot (parity of the tau entry)
        if (it < n_items) {
          const WorkItem wi = item_at(it);
          c->tau[0] = layers[wi.layer].tau_base;
          mbar_arrive_expect_tx(ld_full, step_mode ? 2 * kTileBytes : kTileBytes);
          load2(OB, tmaps + 3 * wi.layer + 1, wi, ld_full);
          if (step_mode) {
            load2(XB, tmaps + 3 * wi.layer + 2, wi, ld_full);
            mbar_arrive_expect_tx(w_full, kTileBytes);
            load2(ST, tmaps + 3 * wi.layer + 0, wi, w_full);
          } else {
            mbar_arrive(w_full);                       // Phi mode: ST is free for the output tile
          }
        }
        for (; it < n_items; it += stride, ++n) {
          const WorkItem wi = item_at(it);
          const long long nxt = it + stride;
          const bool more = nxt < n_items;
          WorkItem wn = wi;
          if (more) {
            wn = item_at(nxt);
            c->tau[(n + 1) & 1] = layers[wn.layer].tau_base;   // read by the epilogue after the next ld_full completes
          }
          if (step_mode) {
            mbar_wait_parked(smem_u32(&c->mp_full), p_mp);    // M' is in XB
            p_mp ^= 1;
            store2(tmaps + 3 * wi.layer + 2, wi, XB);
            tma_wait_group_read0();
            mbar_arrive(smem_u32(&c->xb_free));        // E1 may write Ot into XB
            mbar_wait_parked(smem_u32(&c->xb_mma_free), p_xm);   // the tile's last MMA2 has read XB
            p_xm ^= 1;
            if (more) {
              mbar_arrive_expect_tx(ld_full, 2 * kTileBytes);
              load2(XB, tmaps + 3 * wn.layer + 2, wn, ld_full);
            }
          }
          mbar_wait_parked(smem_u32(&c->ob_mma_free), p_om);  // the tile's last MMA3 has read OB
          p_om ^= 1;
          if (more) {
            if (!step_mode) mbar_arrive_expect_tx(ld_full, kTileBytes);
            load2(OB, tmaps + 3 * wn.layer + 1, wn, ld_full);
          }
          mbar_wait_parked(smem_u32(&c->out_full), p_out);    // W' (Phi mode: the output) is in ST
          p_out ^= 1;
          store2(tmaps + 3 * wi.layer + 0, wi, ST);
          tma_wait_group_read0();
          if (more) {
            if (step_mode) {
              mbar_arrive_expect_tx(w_full, kTileBytes);
              load2(ST, tmaps + 3 * wn.layer + 0, wn, w_full);
            } else {
              mbar_arrive(w_full);
            }
          }
        }
        tma_wait_group0();                             // all stores of this slot have completed
      }
      __syncwarp();
    }
  } else {
    // =================== epilogue warps =========================================================================
    setmaxnreg_inc112();
    const int slot = warp_id >> 3;
    const int ts = tid & (kSlotThreads - 1);
    const int w = warp_id & 7;           // warp of the slot
    const int wq = w & 3;                // TMEM lane quadrant of this warp (= warp index in the CTA mod 4)
    const int h = w >> 2;                // column half: this thread owns the 16-column chunks 2q + h
    const int lane = tid & 31;
    const int t = wq * 32 + lane;        // row of the tile / TMEM lane
    SlotCtrl* sc = &ctrl->slot[slot];
    const uint32_t sb = smem0 + slot * kSlotBytes;
    // Row t of a bf16 buffer: 16-byte chunk ((q & 1) * 4 + 2h + e) ^ (t & 7) of 64-column block q >> 1.  The four
    // chunk offsets a thread ever uses are one XOR apart; keeping them costs 4 registers and no address arithmetic.
    // (`keep`: the value is made opaque to the compiler, which otherwise re-derives such addresses from threadIdx in
    // every phase - 30 % of the instructions of an epilogue - to save the registers.)
    auto keep = [](uint32_t v) { asm volatile("mov.b32 %0, %0;" : "+r"(v)); return v; };
    const uint32_t a0 = sb + (uint32_t)t * 128u + ((((uint32_t)(2 * h)) ^ (uint32_t)(t & 7)) << 4);
    const uint32_t va[4] = {keep(a0), keep(a0 ^ 16u), keep(a0 ^ 64u), keep(a0 ^ 80u)};   // index (q & 1) * 2 + e
    // e4m3 operand row t (one [128 x 128 B] block): 16-byte chunk (2q + h) ^ (t & 7)
    const uint32_t b0 = F8 ? keep(sb + (uint32_t)t * 128u + ((((uint32_t)h) ^ (uint32_t)(t & 7)) << 4)) : 0u;
    auto bf_addr = [&](uint32_t buf, int q, int e) { return va[(q & 1) * 2 + e] + buf + (uint32_t)(q >> 1) * kHalfBytes; };
    const uint32_t opnd_full = smem_u32(&sc->opnd_full), mma_done = smem_u32(&sc->mma_done);
    const uint32_t tmem_slot = tmem_base + slot * kSlotCols;
    const uint32_t lane_off = (uint32_t)(wq * 32) << 16;
    const uint32_t acc_t = keep(tmem_slot + lane_off + 16u * h);
    const uint32_t opa_t = keep(tmem_slot + lane_off + kOpaCol + (F8 ? 4u : 8u) * h);
    // The epilogues work in PIECES of one 16-column chunk: one tcgen05.ld.x16, 8 (bf16) or 4 (e4m3) packed operand
    // words, i.e. two or one 16-byte shared-memory chunks and 8 or 4 TMEM operand columns.  One piece in flight at a
    // time: with the 64-register iterate that is what the 112-register budget holds (a second 16-column buffer to
    // overlap the next load spills 100 B per thread, and a spill here goes to L2: the L1 left beside 205 KB of shared
    // memory does not hold 512 threads' stack frames - measured 34.5 ms; 8-column pieces, double-buffered: 30.4 ms;
    // 16-column pieces, single-buffered: 30.1 ms).
    constexpr int kPC = 16;                   // columns per piece = one 16-column chunk
    constexpr int kNP = 64 / kPC;             // pieces per thread
    constexpr int kXP = kPC / 2;              // packed pairs of the iterate per piece
    constexpr int kW = F8 ? 4 : 8;            // packed operand words per piece
    // piece i = chunk q = i
    auto acc_col = [&](int i) { return 32u * i; };                 // + acc_t
    auto opa_col = [&](int i) { return (F8 ? 8u : 16u) * i; };     // + opa_t
    // the diagonal element of row t: chunk 2 wq + (lane >> 4), i.e. column half lane >> 4, iteration q = wq
    const bool diag_mine = ((lane >> 4) == h);
    const int didx = t & (kPC - 1);

    // The state is Xh = c^(1/4) X: then Ah = Xh Xh^T = sqrt(c) A and B = bA + cA^2 = beta Ah + Ah^2 with
    // beta = b / sqrt(c), so the accumulator after MMA2 is B itself (no rescale in E2).
    const float qs = sqrtf(sqrtf(hp.c));
    const float beta_h = hp.b / sqrtf(hp.c);
    const long long g0 = (long long)blockIdx.x * kSlots + slot;
    int n_my = (int)(n_items > g0 ? (n_items - g0 + stride - 1) / stride : 0);
    uint32_t ph_mma = 0, ph_tile = 0;   // ph_tile: parity of every once-per-tile barrier (ld_full, w_full, xb_free) and of tau[]

    auto load_piece = [&](int i, uint32_t (&c)[kPC]) { tmem_ld16(acc_t + acc_col(i), c); };
    auto pack_piece = [&](const uint32_t (&c)[kPC], float scale, uint32_t (&p)[kW]) {
      if constexpr (F8) pack16_e4m3(c, pk2(scale, scale), p);
      else pack16(c, p);
    };
    auto pack_state = [&](const f2* x, uint32_t (&p)[kW]) {
      if constexpr (F8) {
        const f2 sx2 = pk2(kSX, kSX);
#pragma unroll
        for (int j = 0; j < 4; ++j) p[j] = cvt_e4m3x4(mul2(x[2 * j], sx2), mul2(x[2 * j + 1], sx2));
      } else {
#pragma unroll
        for (int j = 0; j < 8; ++j) p[j] = cvt_bf16x2(x[j]);
      }
    };
    // element didx of the piece (bf16: 16-bit half didx & 1 of word didx >> 1; e4m3: byte didx & 3 of word didx >> 2) := val
    auto patch_diag = [&](uint32_t (&p)[kW], uint32_t val) {
      const uint32_t sh = F8 ? (uint32_t)(didx & 3) * 8u : (uint32_t)(didx & 1) * 16u;
      if constexpr (F8) set_one4(p, didx >> 2, ~(0xffu << sh), val << sh);
      else set_one(p, didx >> 1, ~(0xffffu << sh), val << sh);
    };
    auto store_tmem = [&](int i, const uint32_t (&p)[kW]) {
      if constexpr (F8) tmem_st4(opa_t + opa_col(i), p);
      else tmem_st8(opa_t + opa_col(i), p);
    };
    auto store_operand = [&](uint32_t buf, int i, const uint32_t (&p)[kW]) {
      if constexpr (F8) {
        sts128((b0 ^ ((uint32_t)i << 5)) + buf, make_uint4(p[0], p[1], p[2], p[3]));
      } else {
        sts128(bf_addr(buf, i, 0), make_uint4(p[0], p[1], p[2], p[3]));
        sts128(bf_addr(buf, i, 1), make_uint4(p[4], p[5], p[6], p[7]));
      }
      store_tmem(i, p);
    };
    auto operands_ready = [&](bool wrote_smem) {   // this thread's part of the next product's operands is in place
      tmem_wait_st();
      if (wrote_smem) fence_proxy_async_smem();
      tc_fence_before_sync();
      mbar_arrive(opnd_full);
    };
    auto wait_mma = [&]() {
      mbar_wait_parked(mma_done, ph_mma);
      ph_mma ^= 1;
      tc_fence_after_sync();
    };

    for (; n_my > 0; --n_my, ph_tile ^= 1) {
      // ---------------- P: momentum, normalise ---------------------------------------------------
      TR(0);
      mbar_wait_parked(smem_u32(&sc->ld_full), ph_tile);
      TR(1);
      f2 xs[32];                  // fp32 state: this thread's 4 x 16 columns of row t, as packed pairs (index 8q + 4e + j)
      f2 ss2 = pk2(0.f, 0.f);     // sum of squares of this thread's part of Ghat
      {
        const f2 beta2 = pk2(hp.beta, hp.beta);
#pragma unroll
        for (int i = 0; i < 8; ++i) {              // one 16-byte chunk (8 columns) at a time
          const uint4 gv = lds128(bf_addr(kOB, i >> 1, i & 1));
          const uint32_t gw[4] = {gv.x, gv.y, gv.z, gv.w};
          f2* x = &xs[4 * i];
          if (step_mode) {
            const uint4 mv = lds128(bf_addr(kXB, i >> 1, i & 1));
            const uint32_t mw[4] = {mv.x, mv.y, mv.z, mv.w};
            uint32_t mo[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const f2 g = pk2(bf16_lo(gw[e]), bf16_hi(gw[e]));
              const f2 m = fma2(beta2, pk2(bf16_lo(mw[e]), bf16_hi(mw[e])), g);   // M' = beta M + G
              mo[e] = cvt_bf16x2(m);
              x[e] = hp.nesterov ? fma2(beta2, m, g) : m;                         // Ghat
              ss2 = fma2(x[e], x[e], ss2);
            }
            sts128(bf_addr(kXB, i >> 1, i & 1), make_uint4(mo[0], mo[1], mo[2], mo[3]));   // M' in place
          } else {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              x[e] = pk2(bf16_lo(gw[e]), bf16_hi(gw[e]));
              ss2 = fma2(x[e], x[e], ss2);
            }
          }
        }
      }
      if (step_mode) {
        fence_proxy_async_smem();          // M' in XB -> visible to the TMA store
        mbar_arrive(smem_u32(&sc->mp_full));
      }
      float ss;
      {
        float s0, s1;
        upk2(ss2, s0, s1);
        ss = s0 + s1;
      }
      float tot = ss;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
      if (lane == 0) sc->red[w] = tot;
      named_bar_sync(1 + slot, kSlotThreads);
      TR(2);
      tot = 0.f;
#pragma unroll
      for (int i = 0; i < 8; ++i) tot += sc->red[i];
      const float nrm = sqrtf(tot);
      const float inv = nrm > 0.f ? qs / (nrm + hp.eps) : 0.f;   // Phi_K(0) = 0
      sc->dpart[h][t] = ss * inv * inv;                           // partial diag(Ah)_t in fp32
      {
        const f2 inv2 = pk2(inv, inv);
#pragma unroll
        for (int i = 0; i < kNP; ++i) {
          uint32_t p[kW];
#pragma unroll
          for (int j = 0; j < kXP; ++j) xs[kXP * i + j] = mul2(xs[kXP * i + j], inv2);
          pack_state(&xs[kXP * i], p);
          store_operand(kOB, i, p);
        }
      }
      operands_ready(true);
      TR(4);

      bool dumped = false;   // debug stages: xs holds a raw accumulator dump instead of X_K
      // ---------------- K Newton-Schulz steps ---------------------------------------------------
#pragma unroll 1
      for (int k = 0; k < hp.K; ++k) {
        const bool last = (k + 1 == hp.K);
        // ---- E1: ACC = Ah = Xh Xh^T just landed
        wait_mma();
        TR(10);
        if (kDebugStages && dbg == 1) { dumped = true; break; }
        const float di = sc->dpart[0][t] + sc->dpart[1][t];   // d_t = (Ah)_tt in fp32, from the fp32 state
        if (step_mode && k == 0) mbar_wait_parked(smem_u32(&sc->xb_free), ph_tile);   // the M' store has left XB
        {
          // Ot = offdiag(Ah) + diag(d + beta/2), rounded to the operand format: then for i != j
          //   (Ot Ot^T)_ij = (O^2)_ij + (beta + d_i + d_j) O_ij = (beta Ah + Ah^2)_ij = B_ij.
          uint32_t dval;
          if constexpr (F8) dval = cvt_e4m3x4(pk2(kSO * fmaf(0.5f, beta_h, di), 0.f), pk2(0.f, 0.f)) & 0xffu;
          else dval = pack_bf16(fmaf(0.5f, beta_h, di), 0.f) & 0xffffu;
          f2 Sa = pk2(0.f, 0.f), Sb = Sa;
          uint32_t cc[kPC];
#pragma unroll
          for (int i = 0; i < kNP; ++i) {
            load_piece(i, cc);
            tmem_wait_ld();
#pragma unroll
            for (int j = 0; j < kPC / 4; ++j) {
              const f2 o01 = pk2u(cc[4 * j], cc[4 * j + 1]), o23 = pk2u(cc[4 * j + 2], cc[4 * j + 3]);
              Sa = fma2(o01, o01, Sa);
              Sb = fma2(o23, o23, Sb);
            }
            uint32_t p[kW];
            pack_piece(cc, kSO / (kSX * kSX), p);              // e4m3: ACC = s_X^2 Ah, operand Ot s_O
            if (i == wq) {                                     // warp-uniform: the chunk that holds this warp's diagonal
              if (diag_mine) patch_diag(p, dval);
            }
            store_operand(kXB, i, p);
          }
          float s0, s1;
          upk2(add2(Sa, Sb), s0, s1);
          constexpr float us = F8 ? 1.f / (kSX * kSX) : 1.f;
          sc->spart[h][t] = (s0 + s1) * (us * us);             // partial (Ah^2)_tt
        }
        operands_ready(true);
        TR(13);

        // ---- E2: ACC = B (off-diagonal)
        wait_mma();
        TR(20);
        // a + B_tt, B_tt = beta d_t + (Ah^2)_tt
        const float si = hp.a + fmaf(beta_h, di, sc->spart[0][t] + sc->spart[1][t]);
        if (kDebugStages && dbg == 2) { dumped = true; break; }
        {
          uint32_t cc[kPC];
#pragma unroll
          for (int i = 0; i < kNP; ++i) {
            load_piece(i, cc);
            tmem_wait_ld();
            uint32_t p[kW];
            pack_piece(cc, kSB / (kSO * kSO), p);        // e4m3: ACC = s_O^2 B, operand Bb s_B
            if (i == wq) {
              if (diag_mine) patch_diag(p, 0u);
            }
            store_tmem(i, p);
          }
        }
        operands_ready(false);
        TR(23);

        // ---- E3: Xh = (a + B_tt) Xh + offdiag(B) Xh
        wait_mma();
        TR(30);
        {
          const f2 si2 = pk2(si, si);
          f2 Da = pk2(0.f, 0.f), Db = Da;
          uint32_t cc[kPC];
#pragma unroll
          for (int i = 0; i < kNP; ++i) {
            load_piece(i, cc);
            tmem_wait_ld();
            f2* x = &xs[kXP * i];
            if constexpr (F8) {
              const f2 k3 = pk2(1.f / (kSB * kSX), 1.f / (kSB * kSX));
#pragma unroll
              for (int j = 0; j < kXP; ++j) x[j] = fma2(pk2u(cc[2 * j], cc[2 * j + 1]), k3, mul2(x[j], si2));
            } else {
#pragma unroll
              for (int j = 0; j < kXP; ++j) x[j] = fma2(x[j], si2, pk2u(cc[2 * j], cc[2 * j + 1]));
            }
            if (!last) {
#pragma unroll
              for (int j = 0; j < kXP; j += 2) {
                Da = fma2(x[j], x[j], Da);
                Db = fma2(x[j + 1], x[j + 1], Db);
              }
              uint32_t p[kW];
              pack_state(x, p);
              store_operand(kOB, i, p);
            }
          }
          if (!last) {
            float d0, d1;
            upk2(add2(Da, Db), d0, d1);
            sc->dpart[h][t] = d0 + d1;
          }
        }
        if (!last) operands_ready(true);
        TR(33);
      }
      if (kDebugStages && dumped) {   // tests only: return the raw accumulator instead of X_K
        uint32_t r[kPC];
#pragma unroll
        for (int i = 0; i < kNP; ++i) {
          load_piece(i, r);
          tmem_wait_ld();
#pragma unroll
          for (int j = 0; j < kXP; ++j) xs[kXP * i + j] = pk2u(r[2 * j], r[2 * j + 1]);
        }
        tc_fence_before_sync();
        if (step_mode && dbg == 1) mbar_wait_parked(smem_u32(&sc->xb_free), ph_tile);   // keep the barrier's parity in step
      }
      if (hp.K == 0 && step_mode) mbar_wait_parked(smem_u32(&sc->xb_free), ph_tile);

      // ---------------- F: untile + scaled, weight-decayed write --------------------------------
      TR(40);
      mbar_wait_parked(smem_u32(&sc->w_full), ph_tile);       // W has landed in ST (Phi mode: ST is free)
      TR(41);
      {
        const float keep = 1.f - hp.lr * hp.wd;
        const float unq = dbg ? 1.f : 1.f / qs;                       // undo the c^(1/4) state scaling
        const float stepsz = step_mode ? -hp.lr * hp.scale_c * sc->tau[ph_tile] * unq : unq;
        const f2 step2 = pk2(stepsz, stepsz), keep2 = pk2(keep, keep);
#pragma unroll
        for (int i = 0; i < 8; ++i) {              // one 16-byte chunk (8 columns) at a time
          const f2* x = &xs[4 * i];
          uint32_t p[4];
          if (step_mode) {
            const uint4 wv = lds128(bf_addr(kST, i >> 1, i & 1));
            const uint32_t ww[4] = {wv.x, wv.y, wv.z, wv.w};
#pragma unroll
            for (int e = 0; e < 4; ++e)
              p[e] = cvt_bf16x2(fma2(keep2, pk2(bf16_lo(ww[e]), bf16_hi(ww[e])), mul2(step2, x[e])));
          } else {
#pragma unroll
            for (int e = 0; e < 4; ++e) p[e] = cvt_bf16x2(mul2(step2, x[e]));
          }
          sts128(bf_addr(kST, i >> 1, i & 1), make_uint4(p[0], p[1], p[2], p[3]));
        }
      }
      fence_proxy_async_smem();
      mbar_arrive(smem_u32(&sc->out_full));
      TR(44);
    }
  }


  tc_fence_before_sync();
  __syncthreads();
  if (warp_id == kIssuerWarp) tmem_dealloc<512>(tmem_base);
}

template <bool F8>
cudaError_t launch_t(const LaunchArgs& a, cudaStream_t s, int stage) {
  static DeviceOnce once;   // per device, thread-safe
  cudaError_t e = configure_smem_once(once, himuon_tc128_kernel<F8>, (int)kSmemBytes);
  if (e != cudaSuccess) return e;
  long long grid = (a.n_items + kSlots - 1) / kSlots;
  const int sms = device_sm_count();
  if (grid > sms) grid = sms;
  if (grid < 1) return cudaSuccess;
  himuon_tc128_kernel<F8><<<(unsigned)grid, kThreads, kSmemBytes, s>>>(a.layers, a.tmaps, a.items, a.n_items, a.mode, a.hp, stage);
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_tc128(const LaunchArgs& a, cudaStream_t s) {
#ifdef HIMUON_DEBUG_STAGES
  return launch_t<false>(a, s, g_tc128_debug_stage);
#else
  return launch_t<false>(a, s, 0);
#endif
}
cudaError_t launch_tc128_fp8(const LaunchArgs& a, cudaStream_t s) {
#ifdef HIMUON_DEBUG_STAGES
  return launch_t<true>(a, s, g_tc128_fp8_debug_stage);
#else
  return launch_t<true>(a, s, 0);
#endif
}

}  // namespace himuon

#ifdef HIMUON_DEBUG_STAGES
extern "C" void himuon_debug_set_tc128_stage(int stage) { himuon::g_tc128_debug_stage = stage; }
extern "C" void himuon_debug_set_tc128_fp8_stage(int stage) { himuon::g_tc128_fp8_debug_stage = stage; }
#endif
#ifdef HIMUON_TRACE
extern "C" int himuon_debug_read_trace128(long long* out, int* n) {
  cudaMemcpyFromSymbol(n, himuon::g_tn128, sizeof(int) * 4, 0, cudaMemcpyDeviceToHost);
  return (int)cudaMemcpyFromSymbol(out, himuon::g_trace128, sizeof(long long) * 4 * 16384, 0, cudaMemcpyDeviceToHost);
}
extern "C" int himuon_debug_reset_trace128() {
  int z[4] = {0, 0, 0, 0};
  return (int)cudaMemcpyToSymbol(himuon::g_tn128, z, sizeof(z));
}
#endif
