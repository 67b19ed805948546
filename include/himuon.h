/* himuon.h -- C ABI of the B200-native HiMuon hot path (arxiv/paper_2606_27216).
 *
 * What the library computes (citations are PAPER.md line + section/equation):
 *
 *   Phi_K       K-step quintic Newton-Schulz map                         PAPER.md:63-80, sec. 2.2, Eq. (2.2)-(2.3)
 *                 X_0 = A / (||A||_F + eps);  X_{k+1} = (a I + b X X^T + c (X X^T)^2) X;  Phi_K(0) = 0
 *   B_T, B_T^-1 tiling operator: R = ceil(H/T), C = ceil(W/T), zero padding,
 *               R x C grid of T x T tiles, reassembly + crop             PAPER.md:46-55, sec. 2.1
 *   Phi_{K,T}   Phi_K applied independently to every tile               PAPER.md:126-138, Eq. (4.1)-(4.3)
 *   step        M <- beta M + G;  Ghat = G + beta M (Nesterov) | M;
 *               U = Phi_{K,T}(Ghat);  W <- (1 - lr*wd) W - lr*tau*U;
 *               tau = scale_c*sqrt(T)  (scale_c*sqrt(max(H,W)) if T >= max(H,W))
 *                                                                       PAPER.md:84-105, :153-166, :174-215 (Alg. 4.1), Eq. (4.6)
 *   plan        cross-layer work list of (layer, r, c) tiles, buckets by (T, dtype, path),
 *               memory-bounded chunking (fewest, balanced chunks)       PAPER.md:231-241, sec. 4.4.2-4.4.3, :398
 *
 * Conventions
 *   - Every matrix pointer is a DEVICE pointer owned by the caller (row-major, leading dimension
 *     `ld` in ELEMENTS, ld >= W).  The library never allocates device memory in himuon_step /
 *     himuon_phi / himuon_ns_tiles: all device scratch lives in the caller's `workspace`.
 *   - W and M are updated in place, G is read-only.  Bytes in the `ld - W` gutter are never touched.
 *   - All launches are asynchronous on `cuda_stream` (a cudaStream_t passed as void*; NULL = legacy
 *     default stream).  Host arrays passed in are read before the call returns.
 *   - Errors are return codes; nothing throws across this boundary.  Argument validation happens
 *     before any launch.  There is NO CPU fallback: on a machine without a usable sm_100 device the
 *     compute entry points return HIMUON_ERR_CUDA.
 *   - The plan's work list, buckets and chunks are fixed at himuon_plan_create; the only thing that changes
 *     afterwards is which workspace it is bound to (himuon_plan_bind).  It holds no optimizer state: momentum
 *     lives in the caller's M buffers and survives re-planning with a different T.
 *   - Thread safety: distinct plans may be created, bound and stepped from different host threads and on
 *     different devices concurrently (kernel configuration is per device); one plan is used by one thread
 *     at a time.
 */
#ifndef HIMUON_H_
#define HIMUON_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  HIMUON_OK = 0,
  HIMUON_ERR_INVALID_ARG = 1,        /* null pointer, H/W <= 0, ld < W, K < 0, bad enum, ...              */
  HIMUON_ERR_UNSUPPORTED = 2,        /* valid request this build has no kernel for (see himuon_plan_create) */
  HIMUON_ERR_WORKSPACE_TOO_SMALL = 3,
  HIMUON_ERR_CUDA = 4,               /* a CUDA runtime/driver call failed; see himuon_last_cuda_error()    */
  HIMUON_ERR_NOT_BOUND = 5           /* himuon_step / himuon_phi before himuon_plan_bind                   */
} himuon_status;

typedef enum { HIMUON_F32 = 0, HIMUON_BF16 = 1 } himuon_dtype;

/* Kernel path (PAPER.md:233 buckets tiles by "tile shape, dtype and kernel path").
 *   AUTO : bf16 storage -> tensor-core path (bf16 MMA operands, fp32 accumulation, fp32 X state):
 *            T = 16, 32   one warp per tile, mma.sync, registers only      (any width / ld)
 *            T = 64       tcgen05, two tiles stacked per 128-lane MMA      (W % 8 == 0, ptr and ld*2 16-byte aligned)
 *            T = 128      tcgen05, operands and accumulator in TMEM        (same)
 *            T = 256      tcgen05 cta_group::2, one tile per CTA pair      (same)
 *            T = 512, the full-matrix branch T >= max(H,W) > 256 and rectangular tiles: large-tile path - every
 *                         product of a Newton-Schulz step is one launch of a hand-written persistent tcgen05 GEMM
 *                         (bf16 operands, fp32 accumulation, the iterate as a bf16 hi + lo pair) with the step's elementwise work fused
 *                         into its epilogue; tiles staged in sub-batches inside the caller's workspace
 *                         (himuon_plan_info reports the bytes)
 *          a bf16 matrix whose width is not a multiple of 8 is served by the fp32 kernel at T = 64, 128 and by
 *          the large-tile path at T = 256;
 *          fp32 storage -> fp32 path.
 *   FP32 : true fp32 arithmetic for any storage dtype: FMA kernel for T in {16, 32, 64, 128}; fp32 cuBLAS products
 *          (SGEMM) around fused prep / update kernels for T = 256, 512 and the full-matrix branch (the <= 1e-4 path).
 *   FP8  : bf16 storage, T = 128 or 256, width a multiple of 8 only (anything else: HIMUON_ERR_UNSUPPORTED).  The three
 *          products of a Newton-Schulz step take e4m3 operands (tcgen05 kind::f8f6f4, fp32 accumulation); the
 *          iterate, the diagonals of A and B, momentum and update stay fp32.  Opt-in:
 *          per-tile error about 0.1 instead of <= 3e-2 on Gaussian-like and low-rank tiles, and a heavy-tailed
 *          tile dominated by a few entries (Student-t with 2 degrees of freedom) can leave the basin of the quintic:
 *          the result is then finite but wrong by O(1) or more.  Never selected by AUTO.
 *          Edge tiles with fewer than 32 live rows or columns are run by the bf16 kernel of the same tile size (their
 *          own bucket of the plan, visible through himuon_plan_worklist): too few singular directions to average
 *          e4m3 roundings over. */
typedef enum { HIMUON_PATH_AUTO = 0, HIMUON_PATH_FP32 = 1, HIMUON_PATH_FP8 = 2 } himuon_path;

/* {ptr, H, W, ld, dtype}: one row-major device matrix. */
typedef struct {
  void*   ptr;
  int32_t H, W;
  int64_t ld;        /* elements */
  int32_t dtype;     /* himuon_dtype */
} himuon_mat;

/* One 2-D parameter l of Algorithm 4.1: weight W_l, gradient G_l, momentum M_l (same H, W, dtype).
 * T = 0 selects the plan-wide default; otherwise this layer's tile size (runtime tile schedule).
 * T_w = 0 (or T_w == T): square T x T tiles.  Otherwise rectangular tiles of T rows x T_w columns (PAPER.md:55,
 * the tile-shape study of Fig. 8): both extents powers of two in 16..2048, R = ceil(H/T), C = ceil(W/T_w),
 * tau = scale_c*sqrt(max(T, T_w)); served by the large-tile path (Gram matrix on the short side of
 * the tile): tcgen05 GEMMs on bf16 storage, fp32 cuBLAS products on fp32 storage / HIMUON_PATH_FP32.
 * For himuon_phi only g (input) and w (output) are used; m may be {NULL,...}. */
typedef struct {
  himuon_mat w, g, m;
  int32_t    T;
  int32_t    T_w;
} himuon_layer;

/* Hyper-parameters of Algorithm 4.1 (defaults).
 * (a,b,c) are the Newton-Schulz coefficients; scale_c is the update-scaling constant "c" of
 * sec. 4.2 (the paper uses the letter c for both). eps is ADDED to the Frobenius norm.
 * The tcgen05 kernels (AUTO on bf16 storage at T >= 64, FP8) iterate on c^(1/4) X and need c > 0: with c <= 0
 * (e.g. the cubic iteration (1.5, -0.5, 0)) himuon_step / himuon_phi / himuon_ns_tiles return
 * HIMUON_ERR_UNSUPPORTED before any launch; HIMUON_PATH_FP32, fp32 storage and T = 16, 32 take any finite (a, b, c). */
typedef struct {
  int32_t K;
  float   a, b, c;
  float   eps;
  float   beta;
  int32_t nesterov;
  float   lr, wd, scale_c;
} himuon_hparams;

typedef struct himuon_plan himuon_plan;

/* ---- execution plan (host only) ---------------------------------------- */

/* Build the plan for `n_layers` parameters: enumerate every layer's tiles (layer order of the
 * table, then r-major: index = r*C + c), group them into buckets of equal (T, dtype, path) in
 * order of first appearance, and split each bucket into the fewest balanced chunks such that
 *   fixed_bytes + chunk_tiles * 16  <=  workspace_cap_bytes
 * (16 = one device work item; the fused kernels stage nothing else in HBM).  If the whole list
 * fits it is kept resident and every bucket is one chunk; otherwise chunks are streamed through
 * the workspace one at a time.  workspace_cap_bytes = 0 means "no cap".
 * A layer with T >= max(H,W) is the full-matrix branch: it is run as ONE padded
 * tile of the smallest supported size >= max(H,W) with tau = scale_c*sqrt(max(H,W)); if
 * max(H,W) exceeds the largest tile size (512) it is one whole-matrix item of the large-tile path.
 * Tile sizes: 16, 32, 64, 128, 256, 512 (any T >= max(H,W) selects the full-matrix branch).
 * Tensor-core path needs 16-byte aligned pointers and ld*2 a multiple of 16 (TMA), else
 * HIMUON_ERR_UNSUPPORTED.  Pointers may be NULL when the plan is only inspected (info/worklist);
 * such a plan cannot be bound.  On success *out owns host memory; free with himuon_plan_destroy. */
himuon_status himuon_plan_create(const himuon_layer* layers, int32_t n_layers, int32_t T_default,
                                 int32_t path, size_t workspace_cap_bytes, himuon_plan** out);

/* Sizes of the plan.  Any output pointer may be NULL. */
himuon_status himuon_plan_info(const himuon_plan* plan, int64_t* n_tiles, int32_t* n_buckets,
                               int32_t* n_chunks, size_t* workspace_bytes);

/* Export the work list in execution order: lrc_out[n_tiles][3] = (layer, r, c) and
 * chunk_offsets[n_chunks + 1] (tile index where each chunk starts; last = n_tiles).
 * bucket_T_out[n_chunks] (optional) receives the tile size each chunk runs at. */
himuon_status himuon_plan_worklist(const himuon_plan* plan, int32_t* lrc_out, int64_t* chunk_offsets,
                                   int32_t* bucket_T_out);

/* Memory-bounded chunking rule on its own: fewest chunks with
 * fixed_bytes + items*bytes_per_item <= cap_bytes, balanced sizes (5376 -> 2 x 2688).
 * offsets_out (may be NULL) receives n_chunks+1 entries; returns the number of chunks in *n_chunks. */
himuon_status himuon_plan_chunks(int64_t n_items, int64_t bytes_per_item, int64_t fixed_bytes,
                                 int64_t cap_bytes, int32_t* n_chunks, int64_t* offsets_out,
                                 int32_t offsets_capacity);

/* Copy the plan's device tables (layer table, TMA descriptors, resident work list) into the
 * caller-owned device `workspace` (>= workspace_bytes from himuon_plan_info, 128-byte aligned).
 * Asynchronous on the stream.  Must precede himuon_step / himuon_phi; call again after the
 * workspace moves.  The workspace must stay alive and unmodified while the plan is in use. */
himuon_status himuon_plan_bind(himuon_plan* plan, void* workspace, size_t workspace_bytes,
                               void* cuda_stream);

void himuon_plan_destroy(himuon_plan* plan);

/* ---- compute ------------------------------------------------------------------------------ */

/* One HiMuon optimizer step over every layer of the plan (Algorithm 4.1): one kernel launch per
 * chunk; each launch runs momentum -> tile -> normalise -> K Newton-Schulz steps -> untile ->
 * scaled, weight-decayed parameter write entirely on chip, so every W, G, M element crosses HBM
 * once per direction. */
himuon_status himuon_step(himuon_plan* plan, const himuon_hparams* hp, void* cuda_stream);
/* CUDA graphs: with the plan's work list resident in its workspace (himuon_plan_info: n_chunks chunks all inside the
 * cap, the normal case) himuon_step / himuon_phi enqueue kernel launches only, so after one eager call (which loads
 * and configures the kernels) they may be issued under stream capture and replayed; tests/test_gpu_graph.py.  Not
 * capturable: plans on the fp32 cuBLAS path (T >= 256 on fp32 storage / HIMUON_PATH_FP32) and plans whose work list is
 * streamed chunk by chunk from host memory. */

/* Phi_{K,T} only: w_l <- Phi_{K,T}(g_l) for every layer (no momentum, no scaling; m unused).
 * Uses hp->K, a, b, c, eps only. */
himuon_status himuon_phi(himuon_plan* plan, const himuon_hparams* hp, void* cuda_stream);

/* Packed tiles -> Phi_K(tiles) (sec. 4.4.1; the Fig. 7 workload).
 * tiles_in / tiles_out: device, [n_tiles, T, T] row-major contiguous, edge tiles already
 * zero-padded by the caller (padding stays exactly zero).  In-place allowed.
 * workspace: device, >= himuon_ns_tiles_workspace_bytes(), 128-byte aligned. */
himuon_status himuon_ns_tiles(const void* tiles_in, void* tiles_out, int64_t n_tiles, int32_t T,
                              int32_t dtype, int32_t path, int32_t K, float a, float b, float c,
                              float eps, void* workspace, size_t workspace_bytes, void* cuda_stream);
size_t        himuon_ns_tiles_workspace_bytes(void);

/* himuon_ns_tiles for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): bf16 tiles, HIMUON_PATH_AUTO, same arguments and same result as himuon_ns_tiles
 * (sec. 4.4.1), but WITHOUT a workspace argument.  The device scratch - layer table, tensor maps and,
 * at T = 512, the operand arrays of the large-tile path - is a file-scope `static __device__` array of
 * HIMUON_STATIC_SCRATCH_BYTES inside the library: every GPU that loads the library holds that much device memory
 * until the process exits.  The call issues no cudaMalloc, cudaFree or allocating library routine; it enqueues two
 * small host-to-device copies (the tables) and the kernels on `cuda_stream` and returns.
 *   tiles_in / tiles_out   device, [n_tiles, T, T] bf16 row-major contiguous, 16-byte aligned, caller-owned; in-place
 *                          allowed; edge tiles zero-padded by the caller.
 *   Limit                  the tiles of ONE call must fit the scratch: n_tiles <= himuon_ns_tiles_static_max_tiles(T)
 *                          (T = 512: 12 tiles, 2.5 MiB of operands each; T <= 256 needs no per-tile scratch: 2^31 / T
 *                          tiles).  Beyond it: HIMUON_ERR_WORKSPACE_TOO_SMALL, nothing enqueued, the limit spelled out
 *                          in himuon_last_cuda_error().  fp32 storage and the FP32 / FP8 paths: use himuon_ns_tiles.
 *   Sharing                every call on a device uses the SAME array, which keeps the previous call's contents;
 *                          nothing in it has to start at zero (each call writes every scratch element before reading
 *                          it).  Calls that can overlap on the GPU (different streams, or threads) RACE on it:
 *                          serialise them on one stream or with events.  Other errors as himuon_ns_tiles. */
#define HIMUON_STATIC_SCRATCH_BYTES (32u << 20)
himuon_status himuon_ns_tiles_static(const void* tiles_in, void* tiles_out, int64_t n_tiles, int32_t T, int32_t K,
                                     float a, float b, float c, float eps, void* cuda_stream);
int64_t       himuon_ns_tiles_static_max_tiles(int32_t T);

/* ---- misc --------------------------------------------------------------------------------- */
const char* himuon_status_string(himuon_status s);
/* Text of the last CUDA error seen by this thread's most recent failing call ("" if none). */
const char* himuon_last_cuda_error(void);
/* Bit i set <=> tile size (16 << i) has a kernel on the given path/dtype in this build. */
int32_t     himuon_supported_tile_sizes(int32_t dtype, int32_t path);
/* Number of kernel launches issued by this process through the library (for bench accounting). */
int64_t     himuon_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* HIMUON_H_ */
