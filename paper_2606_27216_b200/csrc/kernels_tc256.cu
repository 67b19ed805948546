// Tensor-core path of the HiMuon hot path for T = 256, bf16 storage: one 256 x 256 tile per CTA PAIR
// (thread-block cluster of 2, tcgen05 cta_group::2), sm_100a.
//
// A 256 x 256 fp32 iterate is 256 KB - the whole register file of an SM - so the tile is split by rows over
// the two CTAs of a cluster: CTA r owns rows 128r .. 128r+127 (its 128 TMEM lanes), keeps them as fp32 in
// registers (64 per thread, 512 threads) and every product of a Newton-Schulz step is ONE
// pair MMA with M = 256 (128 rows per CTA), N = 256, K = 256:
//   the A operand (this CTA's 128 rows x K) is read from this CTA's tensor memory,
//   the B operand (N x K) is split by N: each CTA's shared memory holds 128 of the 256 rows of B,
//   the accumulator (this CTA's 128 rows x 256 columns, fp32) lands in this CTA's tensor memory.
//   MMA1  Ah = Xb Xb^T   B operand = Xb rows (K-major): each CTA contributes its own 128 rows of Xb
//   MMA2  Ot Ot^T        B operand = Ot rows (K-major): likewise
//   MMA3  offdiag(B) Xb  B operand = Xb read MN-major and split by COLUMNS: CTA r must hold columns
//                        128r..128r+127 of all 256 rows, so every thread also writes the bf16 rounding of its
//                        part of the iterate into the owning CTA's staging buffer - half of the threads through
//                        distributed shared memory (st.shared::cluster).  This copy is issued right after MMA1
//                        has been launched, so it overlaps that MMA instead of sitting in an epilogue phase
//                        (measured: 3400 -> 800 cycles for the phase that used to hold it).
// One thread of the leader CTA (rank 0) issues the MMAs once both CTAs have signalled "operands ready" on the
// leader's mbarrier; tcgen05.commit multicasts completion to both CTAs.  Per-tile algorithm, numerical scheme
// and citations: see the header of kernels_tc128.cu (this kernel is its 2-CTA form; same E1/E2/E3 phases).
//
// Every product is issued as TWO N = 128 halves (columns {64 hb..} and {128 + 64 hb..} of the product, hb = 0, 1: a
// cta_group::2 MMA takes half of its N from each CTA), each committed on its own mbarrier, and every thread owns columns
// in both halves - thread (t, q) of a CTA: row t of the CTA's 128 rows (TMEM lane t), the 32-column half q & 1 of the
// 64-column blocks 2 (q >> 1) and 2 (q >> 1) + 1 - so the epilogue of a product starts on the first half while the second
// half still runs on the tensor pipe (a product is seen complete ~500 cycles after its last MMA has been issued,
// that latency is now paid under the first half's epilogue work).  The A operand in tensor
// memory is double-buffered for this: the next product's operand is written while the current one is still read.
// Measured on the Llama-3-8B-shaped step, same box: 61.9 -> 60.4 ms (e4m3 operands 44.3 -> 44.0 ms).
//
// template <bool F8>: the e4m3 variant (HIMUON_PATH_FP8).  Same structure and
// synchronisation; what changes is the operand format of the three products of a Newton-Schulz step: e4m3
// (tcgen05.mma kind::f8f6f4, K = 32 per instruction: 8 instead of 16 MMAs per product, half the operand bytes in shared
// and tensor memory and through distributed shared memory).  Accumulation, the iterate, the diagonals of A and B,
// momentum and update stay fp32.  Operand scales and their justification: header of kernels_tc128.cu (the bounds do
// not depend on T).
#include <cuda_bf16.h>
#include <stddef.h>

#include "himuon_internal.h"
#include "sm100_ptx.cuh"
#include "tc_common.cuh"

namespace himuon {

#ifdef HIMUON_TRACE   // development aid (not built into libhimuon.so): clock stamps of thread 0 of CTA 0
__device__ long long g_trace[2][8192];
__device__ int g_tn;
#define TR() do { if (threadIdx.x == 0 && blockIdx.x == 0 && g_tn < 8192) g_trace[0][g_tn++] = clock64(); } while (0)
#else
#define TR() do { } while (0)
#endif

namespace {

using namespace ptx;
using namespace tc;

constexpr int T = 256;
constexpr int kRows = 128;                       // rows of the tile per CTA
constexpr int kThreads = 512;                    // 16 warps: 4 lane quadrants x 4 column quarters
constexpr uint32_t kBlkBytes = kRows * 128;      // 16 KB: 128 rows x 64 columns bf16 (one swizzle span wide)
constexpr uint32_t kBufBytes = 4 * kBlkBytes;    // 64 KB: 128 rows x 256 columns
constexpr uint32_t kAtomBytes = T * 128;         // 32 KB: 256 K-rows x 64 N-columns (bf16; 128 of e4m3) of the MN-major operand
constexpr float kSX = 256.f, kSO = 128.f, kSB = 128.f;   // e4m3 operand scales (powers of two)
constexpr uint32_t kCtrlBytes = 8192;
constexpr uint32_t kSmemBytes = 3 * kBufBytes + kCtrlBytes + 1024;   // XB, OB, ST + control + alignment slack
constexpr uint32_t kAccCol = 0, kOpaCol = 256;   // TMEM: ACC 256 columns (fp32), 2 x OPA 128 columns (bf16 pairs; e4m3 quads use 64 of each)

struct Ctrl {
  unsigned long long mma_bar[2];  // completion of the two N-halves of a pair product (multicast commit), per CTA
  unsigned long long ready_bar;   // leader CTA only: both CTAs' operands are in place (2 arrivals)
  unsigned long long ld_bar;      // TMA loads of G (and M)
  unsigned long long w_bar;       // TMA load of W
  float dpart[4][kRows];          // per column quarter: partial d_t = sum_j Xh_tj^2
  float spart[4][kRows];          // per column quarter: partial sum_j ACC_tj^2
  float red[16];
  float peer_ss;                  // the other CTA's sum of squares of Ghat
  uint32_t tmem_base;
};
static_assert(sizeof(Ctrl) <= kCtrlBytes, "control block too large");


// K-major operand, this CTA's 128 rows x K = 256: k-step kk = 16 bf16 (32 e4m3) = 32 B inside 128-byte block kk >> 2.
__device__ __forceinline__ uint64_t desc_kmajor(uint32_t buf, int kk) {
  return make_smem_desc_sw128(buf + (kk >> 2) * kBlkBytes + (kk & 3) * 32, 16, 1024);
}
// MN-major operand, K = 256 rows x this CTA's 128 N-columns: bf16 as two 64-column atoms kAtomBytes apart (k-step = 16
// rows of 128 B), e4m3 as one 128-byte span (k-step = 32 rows).
template <bool F8>
__device__ __forceinline__ uint64_t desc_mnmajor(uint32_t buf, int kk) {
  return make_smem_desc_sw128(buf + kk * (F8 ? 4096 : 2048), kAtomBytes, 1024);
}
// One product as two N = 128 halves, each committed on its own barrier so that the epilogue can start on half 0
// while half 1 runs.  A cta_group::2 MMA takes N / 2 rows (columns, MN-major) of B from each CTA: half hb is made
// of B rows 64 hb .. 64 hb + 63 of BOTH CTAs, i.e. the product's columns {64 hb .. +63} and {128 + 64 hb .. +63} -
// global 64-column blocks hb and 2 + hb land in accumulator columns 128 hb .. 128 hb + 127.
template <bool F8>
__device__ __forceinline__ void issue_pair(uint32_t acc, uint32_t opa, uint32_t buf, bool mn_major, uint32_t bar0, uint32_t bar1) {
  const uint32_t idesc = F8 ? (mn_major ? make_idesc_e4m3(T, T / 2, 0, 1) : make_idesc_e4m3(T, T / 2, 0, 0))
                            : (mn_major ? make_idesc_bf16(T, T / 2, 0, 1) : make_idesc_bf16(T, T / 2, 0, 0));
#pragma unroll
  for (int hb = 0; hb < 2; ++hb) {
    // K-major B: 64 rows of 128 B further on; MN-major B: the next 64 columns (bf16: the second atom; e4m3: 64 B on)
    const uint32_t bh = buf + (mn_major ? (F8 ? 64u : kAtomBytes) : 64u * 128u) * hb;
#pragma unroll
    for (int kk = 0; kk < T / (F8 ? 32 : 16); ++kk) {
      const uint64_t db = mn_major ? desc_mnmajor<F8>(bh, kk) : desc_kmajor(bh, kk);
      if (F8) umma_f8_ts_pair(acc + 128 * hb, opa + 8 * kk, db, idesc, kk ? 1u : 0u);
      else umma_bf16_ts_pair(acc + 128 * hb, opa + 8 * kk, db, idesc, kk ? 1u : 0u);
    }
    umma_commit_pair(hb ? bar1 : bar0, (uint16_t)3);
  }
}

template <bool F8>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
himuon_tc256_kernel(const LayerDev* __restrict__ layers, const CUtensorMap* __restrict__ tmaps,
                    const WorkItem* __restrict__ items, long long n_items, int mode, himuon_hparams hp) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
  Ctrl* ctrl = reinterpret_cast<Ctrl*>(smem_raw + (smem0 - smem_u32(smem_raw)) + 3 * kBufBytes);

  const int tid = threadIdx.x;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);   // warp-uniform for the compiler too: the MMA issue stays in uniform registers
  const int wq = warp & 3;             // TMEM lane quadrant of this warp
  const int q4 = warp >> 2;            // column quarter
  const int lane = tid & 31;
  const int t = wq * 32 + lane;        // local row / TMEM lane
  const uint32_t rank = cluster_ctarank();
  const int R = (int)rank * kRows + t; // row of the tile
  const bool lead = (tid == 0);
  const bool step_mode = (mode == MODE_STEP);
  // Column ownership: thread (t, q4) owns the 32-column half s2 = q4 & 1 of the two adjacent global 64-column blocks
  // 2 bp and 2 bp + 1, bp = q4 >> 1, as four 16-column pieces q = 2 hb + j (block 2 bp + hb, chunk j).  Block 2 bp + hb
  // lies in half hb of the accumulator (issue_pair), so every thread has half of its work in each N-half of a product.
  const int s2 = q4 & 1, bp = q4 >> 1;
  // diagonal element (R, R), R = 128 rank + t: block 2 rank + (t >> 6), inner half (t >> 5) & 1, chunk (t >> 4) & 1; bf16:
  // packed word (R & 15) >> 1, half R & 1; e4m3: packed word (R & 15) >> 2, byte R & 3
  const bool own = (q4 == (int)(2 * rank) + (wq & 1));             // warp-uniform
  const int dq = 2 * (wq >> 1) + ((lane >> 4) & 1), dword = F8 ? (t & 15) >> 2 : (t & 15) >> 1;
  const uint32_t dshift = F8 ? (uint32_t)(t & 3) * 8u : (uint32_t)(t & 1) * 16u;
  const uint32_t dkeep = ~((F8 ? 0xffu : 0xffffu) << dshift);

  const uint32_t XB = smem0, OB = XB + kBufBytes, ST = OB + kBufBytes;
  // bf16 rows (operands, and staging of G / M / W): 8-column chunk c = 4 hb + 2 j + e of this thread's 64 columns is
  // 16-byte chunk (4 s2 + (c & 3)) ^ (t & 7) of row t of 64-column block 2 bp + (c >> 2)
  const uint32_t base16 = (uint32_t)(2 * bp) * kBlkBytes + (uint32_t)t * 128u + ((((uint32_t)(4 * s2)) ^ (uint32_t)(t & 7)) << 4);
  auto addr16 = [&](uint32_t buf, int c) { return buf + (base16 ^ ((uint32_t)(c & 3) << 4)) + (uint32_t)(c >> 2) * kBlkBytes; };
  // e4m3 operand rows (first 32 KB of XB / OB): 128-byte block bp of row t, piece q = 16 bytes = chunk 4 hb + 2 s2 + j
  const uint32_t base8 = (uint32_t)bp * kBlkBytes + (uint32_t)t * 128u + ((((uint32_t)(2 * s2)) ^ (uint32_t)(t & 7)) << 4);
  auto addr8 = [&](uint32_t buf, int q) { return buf + (base8 ^ ((uint32_t)(4 * (q >> 1) + (q & 1)) << 4)); };
  // this thread's columns of row R in the MN-major (column-split) copy of Xb, which lives in the staging buffer ST
  // during the steps: both of its blocks belong to CTA bp; K-row R; bf16: atom hb, chunks 4 s2 + 2 j + e of the 128-byte
  // row; e4m3: one 128-byte span per K-row, chunk 4 hb + 2 s2 + j
  const uint32_t xt_local = F8 ? ST + (uint32_t)R * 128u + ((uint32_t)((2 * s2) ^ (R & 7)) << 4)
                               : ST + (uint32_t)R * 128u + ((uint32_t)((4 * s2) ^ (R & 7)) << 4);
  const bool xt_is_local = ((uint32_t)bp == rank);                     // warp-uniform
  const uint32_t xt_row = xt_is_local ? xt_local : mapa_shared(xt_local, (uint32_t)bp);
  auto xt_addr = [&](int q, int e) {
    return F8 ? (xt_row ^ ((uint32_t)(4 * (q >> 1) + (q & 1)) << 4))
              : (xt_row ^ ((uint32_t)(2 * (q & 1) + e) << 4)) + (uint32_t)(q >> 1) * kAtomBytes;
  };
  const uint32_t mma_bar0 = smem_u32(&ctrl->mma_bar[0]), mma_bar1 = smem_u32(&ctrl->mma_bar[1]);
  const uint32_t ready_bar = smem_u32(&ctrl->ready_bar);
  const uint32_t ready_bar_leader = mapa_shared(ready_bar, 0);
  const uint32_t ld_bar = smem_u32(&ctrl->ld_bar);
  const uint32_t w_bar = smem_u32(&ctrl->w_bar);

  if (tid == 0) {
    mbar_init(mma_bar0, 1);
    mbar_init(mma_bar1, 1);
    mbar_init(ready_bar, 2);
    mbar_init(ld_bar, 2);   // arrive.expect_tx at issue + "staging buffer is free" arrive of the lead thread
    mbar_init(w_bar, 1);
    fence_mbar_init();
  }
  cluster_sync_all();                                   // barriers of both CTAs exist before anyone signals
  if (warp == 0) tmem_alloc_pair<512>(smem_u32(&ctrl->tmem_base));
  tc_fence_before_sync();
  cluster_sync_all();
  tc_fence_after_sync();
  const uint32_t tmem_base = ctrl->tmem_base;
  const uint32_t lane_off = (uint32_t)(wq * 32) << 16;
  // piece q = 2 hb + j: accumulator columns 128 hb + 64 bp + 32 s2 + 16 j; operand columns of the global chunk
  // 8 bp + 4 hb + 2 s2 + j (8 packed columns per chunk, e4m3: 4)
  const uint32_t acc_t = tmem_base + lane_off + kAccCol + 64u * bp + 32u * s2;
  const uint32_t opa_t = tmem_base + lane_off + kOpaCol + (F8 ? 4u : 8u) * (8u * bp + 2u * s2);
  auto acc_q = [&](int q) { return acc_t + 128u * (q >> 1) + 16u * (q & 1); };
  auto opa_q = [&](int q) { return opa_t + (F8 ? 4u : 8u) * (4u * (q >> 1) + (q & 1)); };
  const uint32_t ACCd = tmem_base + kAccCol, OPAd = tmem_base + kOpaCol;

  uint32_t ph_mma = 0, ph_ld = 0, ph_w = 0, ph_ready = 0;
  // The A operand is double-buffered in tensor memory (columns 256.. / 384..): an epilogue that starts on the first
  // N-half writes the NEXT product's operand while the second half still reads the current one.
  uint32_t opw = 0;            // column offset (0 / 128) of the operand buffer being written
  const float qs = sqrtf(sqrtf(hp.c));         // state Xh = c^(1/4) X, see kernels_tc128.cu
  const float beta_h = hp.b / sqrtf(hp.c);

  // Operands of the next pair MMA are written: tell the leader; the leader issues once both CTAs have.
  // which: 1 = MMA1 (B = Xb in OB, K-major), 2 = MMA2 (B = Ot in XB, K-major), 3 = MMA3 (B = Xb copy in ST, MN-major).
  auto ready_and_issue = [&](int which) {
    tmem_wait_st();
    // generic-proxy writes -> visible to the MMA.  Remote (DSMEM) writes happen only in write_xb_copy, between the
    // issue of MMA1 and this call for MMA2, so only that call needs the fence over all state spaces.
    // The phase before MMA3 writes tensor memory only.
    if (which == 2) fence_proxy_async_all();
    else if (which == 1) fence_proxy_async_smem();
    tc_fence_before_sync();
    __syncthreads();
    if (warp == 0) {
      if (elect_one()) {
        mbar_arrive_cluster(ready_bar_leader);
        if (rank == 0) {
          mbar_wait_cluster(ready_bar, ph_ready);
          tc_fence_after_sync();
          issue_pair<F8>(ACCd, OPAd + opw, which == 1 ? OB : which == 2 ? XB : ST, which == 3, mma_bar0, mma_bar1);
        }
      }
      __syncwarp();
    }
    ph_ready ^= 1;
    opw ^= 128u;               // the next epilogue writes the other operand buffer
  };
  // N-half hb of the current product is complete (ph_mma flips once per product, after half 1)
  auto wait_mma = [&](int hb) {
    mbar_wait_parked(hb ? mma_bar1 : mma_bar0, ph_mma);
    if (hb) ph_mma ^= 1;
    tc_fence_after_sync();
  };

#ifdef HIMUON_TRACE
  if (threadIdx.x == 0 && blockIdx.x == 0) g_tn = 0;
#endif
  // The column-split bf16 copy of the iterate that MMA3 reads (into ST of the owning CTA).  Called right after
  // MMA1 has been issued, i.e. off the critical path: the stores (half of them remote) overlap the MMA.
  auto write_xb_copy = [&](const f2 (&xs)[32]) {
    const f2 sx2 = pk2(kSX, kSX);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      if (F8) {
        uint32_t x4[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) x4[j] = cvt_e4m3x4(mul2(xs[8 * q + 2 * j], sx2), mul2(xs[8 * q + 2 * j + 1], sx2));
        if (xt_is_local) sts128(xt_addr(q, 0), make_uint4(x4[0], x4[1], x4[2], x4[3]));
        else st_cluster_v4(xt_addr(q, 0), make_uint4(x4[0], x4[1], x4[2], x4[3]));
      } else {
        uint32_t x8[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) x8[j] = cvt_bf16x2(xs[8 * q + j]);
        if (xt_is_local) {
          sts128(xt_addr(q, 0), make_uint4(x8[0], x8[1], x8[2], x8[3]));
          sts128(xt_addr(q, 1), make_uint4(x8[4], x8[5], x8[6], x8[7]));
        } else {
          st_cluster_v4(xt_addr(q, 0), make_uint4(x8[0], x8[1], x8[2], x8[3]));
          st_cluster_v4(xt_addr(q, 1), make_uint4(x8[4], x8[5], x8[6], x8[7]));
        }
      }
    }
  };
  // 16 columns (chunk q of this thread's 64) of the next A operand: rounded to the operand format (e4m3: scaled by
  // `scale` first), the diagonal element replaced by dval when this thread owns it (diag), written to this thread's
  // TMEM operand columns and, if buf is given (XB / OB), to the K-major shared-memory operand in that buffer.
  auto emit_operand = [&](const f2 (&v)[8], f2 scale, int q, bool diag, uint32_t dval, uint32_t buf) {
    if (F8) {
      uint32_t p[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) p[j] = cvt_e4m3x4(mul2(v[2 * j], scale), mul2(v[2 * j + 1], scale));
      if (diag) set_one4(p, dq == q ? dword : 4, dkeep, dval);
      if (buf) sts128(addr8(buf, q), make_uint4(p[0], p[1], p[2], p[3]));
      tmem_st4(opa_q(q) + opw, p);
    } else {
      uint32_t p[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) p[j] = cvt_bf16x2(v[j]);
      if (diag) set_one(p, dq == q ? dword : 8, dkeep, dval);
      if (buf) {
        sts128(addr16(buf, 2 * q), make_uint4(p[0], p[1], p[2], p[3]));
        sts128(addr16(buf, 2 * q + 1), make_uint4(p[4], p[5], p[6], p[7]));
      }
      tmem_st8(opa_q(q) + opw, p);
    }
  };
  auto acc_pairs = [](const uint32_t (&c)[16], f2 (&v)[8]) {
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = pk2u(c[2 * j], c[2 * j + 1]);
  };

  // G -> OB and (step mode) M -> XB of tile i: this CTA's 128 rows, four 64-column boxes each
  auto issue_gm = [&](long long i) {
    WorkItem wn;
    if (items) wn = items[i];
    else { wn.layer = 0; wn.r = (int)i; wn.c = 0; wn.pad = 0; }
    const int xn = wn.c * T, yn = wn.r * T + (int)rank * kRows;
    mbar_arrive_expect_tx(ld_bar, step_mode ? 2 * kBufBytes : kBufBytes);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      tma_load_2d(OB + j * kBlkBytes, tmaps + 3 * wn.layer + 1, xn + 64 * j, yn, ld_bar);
      if (step_mode) tma_load_2d(XB + j * kBlkBytes, tmaps + 3 * wn.layer + 2, xn + 64 * j, yn, ld_bar);
    }
  };
  bool prefetched = false;   // every thread tracks it (uniform); only the lead thread issues

  for (long long it = cluster_id_x(); it < n_items; it += cluster_count_x()) {
    TR();   // tile start
    WorkItem wi;
    if (items) wi = items[it];
    else { wi.layer = 0; wi.r = (int)it; wi.c = 0; wi.pad = 0; }
    const float tau_base = layers[wi.layer].tau_base;
    const CUtensorMap* map_w = tmaps + 3 * wi.layer + 0;
    const CUtensorMap* map_m = tmaps + 3 * wi.layer + 2;
    const int x0 = wi.c * T, y0 = wi.r * T + (int)rank * kRows;
    bool w_issued = false;
    const long long nxt = it + cluster_count_x();

    // ---------------- P: load, momentum, normalise ---------------------------------------------------
    if (lead) {
      if (!prefetched) issue_gm(it);
      mbar_arrive(ld_bar);
    }
    mbar_wait(ld_bar, ph_ld);
    ph_ld ^= 1;
    prefetched = false;
    TR();   // G, M landed and the staging buffer is free

    f2 xs[32];                  // fp32 state: this thread's 64 columns of row R, as packed pairs
    f2 ss2 = pk2(0.f, 0.f);
    const f2 beta2 = pk2(hp.beta, hp.beta);
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      const uint4 gv = lds128(addr16(OB, c));
      const uint32_t gw[4] = {gv.x, gv.y, gv.z, gv.w};
      if (step_mode) {
        const uint4 mv = lds128(addr16(XB, c));
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
        sts128(addr16(XB, c), make_uint4(mo[0], mo[1], mo[2], mo[3]));   // M' in place, over this thread's M
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
    if (lane == 0) ctrl->red[warp] = tot;
    fence_proxy_async_smem();          // M' in XB -> visible to the TMA store
    __syncthreads();
    TR();   // momentum pass done
    float mine = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) mine += ctrl->red[i];
    if (lead) {
      // M' leaves from XB, where it was computed in place: nothing waits for that store here (XB is next written
      // by E1 of the first step, thousands of cycles later).  What must have drained before the cluster barrier
      // below is the PREVIOUS tile's store out of ST: after the barrier ST of BOTH CTAs may receive the Xb copy.
      // (A TMA store of 64 KB takes ~3000 cycles to drain at this SM's share of the HBM write bandwidth.  Writing
      // W' to global memory straight from the registers instead, with no store pending on ST, was measured too:
      // 66.0 ms against 62.2 ms - the LSU store path costs more than the drain.)
      if (step_mode) {
#pragma unroll
        for (int j = 0; j < 4; ++j) tma_store_2d(map_m, x0 + 64 * j, y0, XB + j * kBlkBytes);
        tma_commit_group();
        tma_wait_group_read1();
      } else {
        tma_wait_group_read0();
      }
      st_cluster_f32(mapa_shared(smem_u32(&ctrl->peer_ss), rank ^ 1u), mine);   // Frobenius norm spans both CTAs
    }
    cluster_sync_all();
    TR();   // M' on its way, norm exchanged
    tot = mine + ctrl->peer_ss;
    const float nrm = sqrtf(tot);
    const float inv = nrm > 0.f ? qs / (nrm + hp.eps) : 0.f;   // Phi_K(0) = 0
    ctrl->dpart[q4][t] = ss * inv * inv;                        // partial diag(Ah)_R in fp32
    {
      const f2 inv2 = pk2(inv, inv), sx2 = pk2(kSX, kSX);
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        f2 v[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = xs[8 * q + j] = mul2(xs[8 * q + j], inv2);
        emit_operand(v, sx2, q, false, 0u, OB);   // Xb lives in OB (G is consumed), Ot in XB: see the M' store above
      }
    }
    TR();   // prologue compute done
    if (hp.K > 0) ready_and_issue(1);
    else __syncthreads();
    TR();   // MMA1 issued
    if (hp.K > 0) write_xb_copy(xs);
    float di = (ctrl->dpart[0][t] + ctrl->dpart[1][t]) + (ctrl->dpart[2][t] + ctrl->dpart[3][t]);

    // ---------------- K Newton-Schulz steps ---------------------------------------------------
#pragma unroll 1
    for (int k = 0; k < hp.K; ++k) {
      const bool last = (k + 1 == hp.K);
      // ---- E1: ACC = rows of Ah
      if (k == 0 && step_mode) {                                 // M' has left XB (long ago): Ot may be written into it
        if (lead) tma_wait_group_read0();
        __syncthreads();
      }
      wait_mma(0);
      TR();   // MMA1 done (first half)
      {
        // Ot = offdiag(Ah) + diag(d + beta/2), rounded to bf16: offdiag(Ot Ot^T) = offdiag(beta Ah + Ah^2)
        // (e4m3: ACC = s_X^2 Ah; operand scale s_O: Ot s_O = ACC s_O / s_X^2)
        const float dv = fmaf(0.5f, beta_h, di);
        const uint32_t dval = F8 ? (cvt_e4m3x4(pk2(kSO * dv, 0.f), pk2(0.f, 0.f)) & 0xffu) << dshift
                                 : (pack_bf16(dv, 0.f) & 0xffffu) << dshift;
        const f2 k1 = pk2(kSO / (kSX * kSX), kSO / (kSX * kSX));
        f2 Sa = pk2(0.f, 0.f), Sb = Sa;
        uint32_t r[2][16];
        tmem_ld16(acc_q(0), r[0]);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          tmem_wait_ld();
          if (q != 1 && q < 3) tmem_ld16(acc_q(q + 1), r[(q + 1) & 1]);
          uint32_t(&c)[16] = r[q & 1];
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const f2 o01 = pk2u(c[4 * j], c[4 * j + 1]), o23 = pk2u(c[4 * j + 2], c[4 * j + 3]);
            Sa = fma2(o01, o01, Sa);
            Sb = fma2(o23, o23, Sb);
          }
          f2 v[8];
          acc_pairs(c, v);
          emit_operand(v, k1, q, own, dval, XB);
          if (q == 1) {                              // pieces 2, 3 live in the second N-half
            wait_mma(1);
            tmem_ld16(acc_q(2), r[0]);
          }
        }
        float s0, s1;
        upk2(add2(Sa, Sb), s0, s1);
        const float us = F8 ? 1.f / (kSX * kSX) : 1.f;         // partial (Ah^2)_RR (e4m3: from the scaled accumulator)
        ctrl->spart[q4][t] = (s0 + s1) * (us * us);
      }
      TR();   // E1 loop done
      ready_and_issue(2);
      TR();   // MMA2 issued
      // a + B_RR, B_RR = beta d_R + (Ah^2)_RR
      const float si = hp.a + fmaf(beta_h, di, (ctrl->spart[0][t] + ctrl->spart[1][t]) + (ctrl->spart[2][t] + ctrl->spart[3][t]));

      // ---- E2: ACC = rows of B (off-diagonal)
      wait_mma(0);
      TR();   // MMA2 done (first half)
      {
        uint32_t r[2][16];
        tmem_ld16(acc_q(0), r[0]);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          tmem_wait_ld();
          if (q != 1 && q < 3) tmem_ld16(acc_q(q + 1), r[(q + 1) & 1]);
          f2 v[8];
          acc_pairs(r[q & 1], v);
          emit_operand(v, pk2(kSB / (kSO * kSO), kSB / (kSO * kSO)), q, own, 0u, 0u);   // e4m3: ACC = s_O^2 B; operand Bb s_B
          if (q == 1) {
            wait_mma(1);
            tmem_ld16(acc_q(2), r[0]);
          }
        }
      }
      TR();   // E2 loop done
      ready_and_issue(3);
      TR();   // MMA3 issued

      // ---- E3: Xh = (a + B_RR) Xh + offdiag(B) Xh
      wait_mma(0);
      TR();   // MMA3 done (first half)
      auto after_last_mma = [&]() {
        if (last && lead && step_mode) {                     // ST is free (every pair MMA has completed): fetch W into
          mbar_arrive_expect_tx(w_bar, kBufBytes);           // it - FIRST, phase F needs it long before P needs G, M
#pragma unroll
          for (int j = 0; j < 4; ++j) tma_load_2d(ST + j * kBlkBytes, map_w, x0 + 64 * j, y0, w_bar);
          w_issued = true;
        }
        if (last && nxt < n_items) {                         // ... and so are XB and OB: the next tile's G and M
          if (lead) issue_gm(nxt);
          prefetched = true;
        }
      };
      {
        const f2 si2 = pk2(si, si), k3 = pk2(1.f / (kSB * kSX), 1.f / (kSB * kSX)), sx2 = pk2(kSX, kSX);
        f2 Da = pk2(0.f, 0.f), Db = Da;
        uint32_t r[2][16];
        tmem_ld16(acc_q(0), r[0]);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          tmem_wait_ld();
          if (q != 1 && q < 3) tmem_ld16(acc_q(q + 1), r[(q + 1) & 1]);
          uint32_t(&c)[16] = r[q & 1];
#pragma unroll
          for (int j = 0; j < 8; ++j)
            xs[8 * q + j] = F8 ? fma2(pk2u(c[2 * j], c[2 * j + 1]), k3, mul2(xs[8 * q + j], si2))
                               : fma2(xs[8 * q + j], si2, pk2u(c[2 * j], c[2 * j + 1]));
          if (!last) {
#pragma unroll
            for (int j = 0; j < 8; j += 2) {
              Da = fma2(xs[8 * q + j], xs[8 * q + j], Da);
              Db = fma2(xs[8 * q + j + 1], xs[8 * q + j + 1], Db);
            }
            f2 v[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) v[j] = xs[8 * q + j];
            emit_operand(v, sx2, q, false, 0u, OB);
          }
          if (q == 1) {
            wait_mma(1);
            after_last_mma();
            tmem_ld16(acc_q(2), r[0]);
          }
        }
        if (!last) {
          float d0, d1;
          upk2(add2(Da, Db), d0, d1);
          ctrl->dpart[q4][t] = d0 + d1;
        }
      }
      TR();   // E3 loop done
      if (!last) {
        ready_and_issue(1);
        write_xb_copy(xs);
        di = (ctrl->dpart[0][t] + ctrl->dpart[1][t]) + (ctrl->dpart[2][t] + ctrl->dpart[3][t]);
      } else {
        tc_fence_before_sync();
      }
      TR();   // MMA1 of the next step issued (or nothing)
    }

    // ---------------- F: untile + scaled, weight-decayed write --------------------------------
    if (step_mode) {
      if (lead && !w_issued) {                               // K = 0: W was not prefetched
        tma_wait_group_read0();
        mbar_arrive_expect_tx(w_bar, kBufBytes);
#pragma unroll
        for (int j = 0; j < 4; ++j) tma_load_2d(ST + j * kBlkBytes, map_w, x0 + 64 * j, y0, w_bar);
      }
      mbar_wait(w_bar, ph_w);
      ph_w ^= 1;
    } else {
      if (lead) tma_wait_group_read0();                      // Phi mode: the previous output has left ST
      __syncthreads();
    }
    TR();   // W landed
    {
      const float keep = 1.f - hp.lr * hp.wd;
      const float unq = 1.f / qs;                                   // undo the c^(1/4) state scaling
      const float stepsz = step_mode ? -hp.lr * hp.scale_c * tau_base * unq : unq;
      const f2 step2 = pk2(stepsz, stepsz), keep2 = pk2(keep, keep);
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        uint32_t p[4];
        if (step_mode) {
          const uint4 wv = lds128(addr16(ST, c));
          const uint32_t ww[4] = {wv.x, wv.y, wv.z, wv.w};
#pragma unroll
          for (int e = 0; e < 4; ++e)
            p[e] = cvt_bf16x2(fma2(keep2, pk2u(ww[e] << 16, ww[e] & 0xffff0000u), mul2(step2, xs[4 * c + e])));
        } else {
#pragma unroll
          for (int e = 0; e < 4; ++e) p[e] = cvt_bf16x2(mul2(step2, xs[4 * c + e]));
        }
        sts128(addr16(ST, c), make_uint4(p[0], p[1], p[2], p[3]));
      }
    }
    fence_proxy_async_smem();
    __syncthreads();
    if (lead) {
#pragma unroll
      for (int j = 0; j < 4; ++j) tma_store_2d(map_w, x0 + 64 * j, y0, ST + j * kBlkBytes);
      tma_commit_group();
    }
  }

  if (lead) tma_wait_group0();
  tc_fence_before_sync();
  cluster_sync_all();
  if (warp == 0) tmem_dealloc_pair<512>(tmem_base);
}

}  // namespace

namespace {
template <bool F8>
cudaError_t launch_tc256_t(const LaunchArgs& a, cudaStream_t s) {
  static DeviceOnce once;   // per device, thread-safe
  cudaError_t e = configure_smem_once(once, himuon_tc256_kernel<F8>, (int)kSmemBytes);
  if (e != cudaSuccess) return e;
  if (a.n_items < 1) return cudaSuccess;
  long long clusters = a.n_items;
  const int max_clusters = device_sm_count() / 2;
  if (clusters > max_clusters) clusters = max_clusters;
  himuon_tc256_kernel<F8><<<(unsigned)(2 * clusters), kThreads, kSmemBytes, s>>>(a.layers, a.tmaps, a.items, a.n_items, a.mode, a.hp);
  return cudaGetLastError();
}
}  // namespace
cudaError_t launch_tc256(const LaunchArgs& a, cudaStream_t s) { return launch_tc256_t<false>(a, s); }
cudaError_t launch_tc256_fp8(const LaunchArgs& a, cudaStream_t s) { return launch_tc256_t<true>(a, s); }

}  // namespace himuon

#ifdef HIMUON_TRACE
extern "C" int himuon_debug_read_trace(long long* out, int n) {
  return (int)cudaMemcpyFromSymbol(out, himuon::g_trace, sizeof(long long) * (size_t)n, 0, cudaMemcpyDeviceToHost);
}
#endif
