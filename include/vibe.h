/* vibe.h -- C ABI of libvibe.so: the B200-native (sm_100a) per-GPU MoE-layer hot path
 * behind ViBE's variability-aware expert placement (arxiv 2606.00735).
 *
 * Citations: P:L<n> = PAPER.md line n (ViBE paper).  Reading ids (R1.., P1.., F1..,
 * M1.., L1..) are listed in DESIGN.md "Readings of the paper".  The paper treats the
 * per-GPU MoE layer ("the fused MoE kernel") as a black box that it
 * profiles as latency-vs-token-load f_g(n) and counts expert activations for
 * (activation matrix W).  This library IS that black box, rebuilt for one B200:
 *
 *   vibe_route_topk   -> vibe_permute -> vibe_grouped_ffn -> vibe_combine       (one stream,
 *   no host synchronisation between calls), plus vibe_profile_expert_latency which measures
 *   f(n), and the host-side placement evaluator / greedy solver that consume it
 *   (Algorithm 1 Phase 2 P:L446-L453).
 *
 * Conventions
 *   - Plain C, no torch / C++ types.  Every pointer is a DEVICE pointer unless the
 *     parameter comment says "host".  bf16 tensors are passed as `const void*` to raw
 *     16-bit storage; all tensors are dense row-major.
 *   - The caller owns every buffer, including workspaces (size them with
 *     vibe_workspace_bytes / vibe_rows_cap).  The library allocates no device memory per
 *     call; it keeps process-lifetime caches only (TMA tensor maps keyed by pointer+shape).
 *   - All device work is enqueued asynchronously on `stream` (a cudaStream_t passed as
 *     void*; NULL = legacy default stream).  No call synchronises with the host except
 *     vibe_profile_expert_latency and vibe_moe_layer_forward_host (they return host data).
 *   - Data-dependent sizes (rows per expert) are never read back: kernels take extents
 *     from the device-side `offsets` array.
 *   - Errors: every function returns a vibe_status; argument errors are detected before
 *     any launch; text of the last error on this thread: vibe_last_error().
 *   - There is no CPU fallback and no other back-end.  Without a CUDA device every compute
 *     entry point returns VIBE_ERR_CUDA.
 *   - Inputs must be finite.  NaN/Inf behaviour is unspecified.
 */
#ifndef VIBE_H_
#define VIBE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(_WIN32)
#define VIBE_API
#else
#define VIBE_API __attribute__((visibility("default")))
#endif

typedef enum {
  VIBE_OK = 0,
  VIBE_ERR_INVALID_ARG = 1, /* null pointer, bad size, inconsistent config          */
  VIBE_ERR_UNSUPPORTED = 2, /* valid request outside what the kernels implement      */
  VIBE_ERR_WORKSPACE = 3,   /* workspace pointer null / too small / misaligned       */
  VIBE_ERR_CUDA = 4         /* CUDA runtime / driver error (text in vibe_last_error) */
} vibe_status;

typedef enum { VIBE_SCORE_SOFTMAX = 0, VIBE_SCORE_SIGMOID = 1 } vibe_score_fn;

/* Routing configuration (readings R1-R7).  Plain data, host memory. */
typedef struct {
  int32_t num_experts;      /* E: global experts, 1..512                                  */
  int32_t top_k;            /* k: 1..min(E,32)                                            */
  int32_t score_fn;         /* vibe_score_fn                                              */
  int32_t renormalize;      /* 1: divide the k gate weights by their sum (no epsilon, R4) */
  float routed_scale;       /* multiplies the final weights (R5); 1.0f in all configs     */
  int32_t n_group;          /* 0 or 1: no group limiting; else E % n_group == 0 (R6)      */
  int32_t topk_group;       /* groups kept; topk_group * (E/n_group) >= k                 */
  const float* select_bias; /* DEVICE [E] or NULL: added to the score for SELECTION only  */
} vibe_route_cfg;

/* ------------------------------------------------------------------------------------
 * a1 + a2.  Top-k routing with fused expert-activation histogram.
 * "route each token to a subset of experts"; counts = one row of the
 * activation matrix W in R^{LxE}, over GLOBAL experts (R8).
 *
 * Per token t (readings R1-R3, R6):
 *   key[e]  = logits[t,e]                               (softmax: select on raw logits)
 *           = vsig(logits[t,e]) + select_bias[e]        (sigmoid; vsig = the fixed sequence
 *             of correctly rounded binary32 operations given in DESIGN.md R2, so ids are
 *             reproducible bit for bit)
 *   group limiting: E/n_group contiguous experts per group, group score = largest +
 *             second largest key (one f32 add), keep the topk_group best groups
 *             (ties -> lower group), other keys = -inf
 *   topk_ids[t,0..k) = k rounds of arg-max, ties -> LOWEST expert index, in pick order
 *   topk_w[t,j]      = softmax over all E of logits (or the true sigmoid, bias excluded) at
 *             the picked experts, evaluated in fp64, optionally renormalised over the k
 *             picks, times routed_scale, rounded once to f32
 *   counts[e]        = number of (t,j) with topk_ids[t,j] == e   (overwritten, not accumulated)
 *
 * logits [T,E] f32 (16-byte aligned), topk_ids [T,k] i32, topk_w [T,k] f32, counts [E] i32.
 * T >= 0 (T == 0 just zeroes counts).  T*k < 2^31.
 * ---------------------------------------------------------------------------------- */
VIBE_API vibe_status vibe_route_topk(const vibe_route_cfg* cfg /*host*/, const float* logits, int32_t T,
                                     int32_t* topk_ids, float* topk_w, int32_t* counts, void* stream);

/* ------------------------------------------------------------------------------------
 * a3.  Permute: stable counting sort of the A = T*k assignments (flat index i = t*k+j) by
 * local expert slot, and gather of the token rows into expert-contiguous order.
 * "token dispatch remains local"; readings P1-P4.
 *
 *   slot(i)   = expert_map[topk_ids[i]]  (-1 = expert not resident on this GPU)
 *   offsets[0] = 0; offsets[s+1] = offsets[s] + roundup(#{i: slot(i)=s}, align)
 *   rows of slot s are its assignments in ascending i (stable); then padding rows
 *   row_to_assign[r] = i (or -1 for padding); assign_to_row[i] = r (or -1 if not resident)
 *   Xp[r,:] = X[i / k, :] (bit copy); padding rows are zero
 * Rows >= offsets[E_loc] are not written.
 *
 * X [T,d] bf16; expert_map [E] i32 or NULL (identity, requires E_loc == E);
 * d % 8 == 0 (16-byte rows); align >= 1.
 * Outputs: Xp [R_cap,d] bf16, offsets [E_loc+1] i32, row_to_assign [R_cap] i32,
 * assign_to_row [A] i32, with R_cap >= vibe_rows_cap(T,k,E_loc,align).
 * counts: optional (may be NULL) -- the histogram produced by vibe_route_topk; advisory.
 * ws: vibe_workspace_bytes(VIBE_WS_PERMUTE, ...) bytes, 16-byte aligned; scratch of THIS call (a table of
 *     per-CTA slot totals and the grid-barrier counters): calls that may run concurrently -- other streams,
 *     graphs replayed side by side -- must be given different workspaces.
 * ---------------------------------------------------------------------------------- */
VIBE_API vibe_status vibe_permute(const void* X, const int32_t* topk_ids, const int32_t* counts,
                                  const int32_t* expert_map, int32_t T, int32_t d, int32_t k, int32_t E,
                                  int32_t E_loc, int32_t align, void* Xp, int32_t* offsets,
                                  int32_t* row_to_assign, int32_t* assign_to_row, void* ws, size_t ws_bytes,
                                  void* stream);

/* a3 without a workspace argument, for callers that cannot allocate device memory (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): the same operation, arguments, layouts and results as
 * vibe_permute (readings P1-P4; /root/reference PAPER.md L28, L86: tokens are sent to their experts), with
 * the scratch of the index kernel in a static device array of VIBE_PERMUTE_STATIC_BYTES inside the library (every GPU
 * that loads the library holds it until the process exits).  The call allocates nothing (no cudaMalloc / cudaFree /
 * allocating library routine).
 * Limit: vibe_workspace_bytes(VIBE_WS_PERMUTE, ...) = roundup(4 * SMs * E_loc, 256) + 256 bytes must fit the array:
 *   E_loc <= 512 on a 148-SM B200; beyond that VIBE_ERR_WORKSPACE (nothing is launched; use vibe_permute).
 * ALL calls of a process on one GPU share the array: calls that may overlap on the GPU (different streams, graphs
 * replayed side by side) race on it and must use vibe_permute with their own workspaces instead.  The array keeps
 * the last call's contents; every call clears what it needs cleared.  Other errors: as vibe_permute. */
#define VIBE_PERMUTE_STATIC_BYTES (304 * 1024)
VIBE_API vibe_status vibe_permute_static(const void* X, const int32_t* topk_ids, const int32_t* counts,
                                         const int32_t* expert_map, int32_t T, int32_t d, int32_t k, int32_t E,
                                         int32_t E_loc, int32_t align, void* Xp, int32_t* offsets,
                                         int32_t* row_to_assign, int32_t* assign_to_row, void* stream);

/* ------------------------------------------------------------------------------------
 * a4.  Grouped SwiGLU expert FFN over the resident experts -- the kernel whose
 * latency-vs-token-load ViBE profiles and the dominant cost of MoE serving
 * (49 % of prefill time).  Readings F1-F4.
 *
 *   for slot s, rows r in [offsets[s], offsets[s+1]):
 *     H[r,:] = bf16( silu(Xp[r,:] . W1[s]) * (Xp[r,:] . W3[s]) )      (fp32 accumulate)
 *     Y[r,:] = bf16( H[r,:] . W2[s] )                                  (fp32 accumulate)
 *
 * Xp [R_cap,d] bf16; offsets [E_loc+1] i32 (device; offsets[E_loc] <= R_cap);
 * W1, W3 [E_loc,d,f] bf16 (gate, up); W2 [E_loc,f,d] bf16 (down); all row-major, consumed
 * in place (no repacking).  H_ws [R_cap,f] bf16 scratch; Y [R_cap,d] bf16.
 * Shape limits of the tcgen05 kernels: d % 64 == 0, f % 64 == 0, all base pointers
 * 16-byte aligned (TMA), R_cap >= 1.  Rows >= offsets[E_loc] of H_ws / Y are not written.
 * ws: vibe_workspace_bytes(VIBE_WS_FFN, ...) bytes, 16-byte aligned, or NULL.  It holds the fp32 partial sums and the
 *     arrival counters of the SPLIT-K path: when a launch has at most half as many tiles as the GPU
 *     has CTA pairs -- a lone or a few light experts, the decode regime P:L108 / L130 calls low-intensity -- every
 *     tile's K range is cut over several pairs and reduced in fp32 in a fixed order.  With ws = NULL (or too small)
 *     the call is still correct; such launches then stream their weights on as many SM pairs as they have tiles.
 *     The workspace also holds the unit counters of the DYNAMIC tile hand-out used for long-K launches (the CTA pairs
 *     take the next tile from one counter when they are ready, so that the token tiles sharing a weight tile run
 *     together and share it through L2: DRAM traffic 1.08 x instead of 1.5 x the algorithmic bytes at the C1 shape);
 *     without a workspace tiles are assigned statically.  Results do not depend on the workspace being given beyond
 *     the fp32 summation order of split tiles, and are bit-reproducible from call to call either way.
 *     Calls that may run concurrently must use different workspaces.
 * ---------------------------------------------------------------------------------- */
VIBE_API vibe_status vibe_grouped_ffn(const void* Xp, const int32_t* offsets, int32_t E_loc, int32_t R_cap,
                                      int32_t d, int32_t f, const void* W1, const void* W3, const void* W2,
                                      void* H_ws, void* Y, void* ws, size_t ws_bytes, void* stream);

/* ------------------------------------------------------------------------------------
 * a5.  Weighted un-permute / combine (reading C1):
 *   out[t,:] = bf16( sum_{j<k, assign_to_row[t*k+j] >= 0} topk_w[t,j] * Y[assign_to_row[t*k+j],:] )
 * fp32 accumulation in slot order j = 0..k-1 (deterministic); tokens without a resident
 * expert get zeros.  Y [R_cap,d] bf16, out [T,d] bf16, d % 8 == 0.
 * ---------------------------------------------------------------------------------- */
VIBE_API vibe_status vibe_combine(const void* Y, const int32_t* assign_to_row, const float* topk_w, int32_t T,
                                  int32_t k, int32_t d, void* out, void* stream);

/* ------------------------------------------------------------------------------------
 * a4 + a5 fused ("gate-weighted scatter fused into the down projection", BJ:north_star).
 * vibe_grouped_ffn_scatter computes the same FFN as vibe_grouped_ffn, but the epilogue of the
 * down projection multiplies row r by the gate weight of its assignment i = row_to_assign[r]
 * and stores it at row i of Yw -- Yw [T*k, d] bf16 is in ASSIGNMENT order:
 *     Yw[i,:] = bf16( topk_w[i] * y(assign_to_row[i]) )        (one rounding of the product)
 * Rows of non-resident assignments are NOT written.  vibe_combine_scattered then reduces k
 * CONTIGUOUS rows per token:  out[t,:] = bf16( sum_{j: assign_to_row[t*k+j] >= 0} Yw[t*k+j,:] ),
 * fp32, slot order.  Same layouts, ownership and errors as vibe_grouped_ffn / vibe_combine.
 * ---------------------------------------------------------------------------------- */
VIBE_API vibe_status vibe_grouped_ffn_scatter(const void* Xp, const int32_t* offsets, int32_t E_loc,
                                              int32_t R_cap, int32_t d, int32_t f, const void* W1,
                                              const void* W3, const void* W2, const int32_t* row_to_assign,
                                              const float* topk_w, void* H_ws, void* Yw, void* ws,
                                              size_t ws_bytes, void* stream);
VIBE_API vibe_status vibe_combine_scattered(const void* Yw, const int32_t* assign_to_row, int32_t T, int32_t k,
                                            int32_t d, void* out, void* stream);

/* ------------------------------------------------------------------------------------
 * f2.  The grouped FFN with FP8 (e4m3) operands -- "Precision: FP8" for both evaluated
 * models (Table 2a); the recipe is DESIGN.md readings Q1-Q4:
 *   e4m3 = OCP FP8 E4M3 (no infinities, max 448), round-to-nearest-even, saturating;
 *   scale = binary32(absmax / 448), 1 for an all-zero row / expert; code = e4m3(binary32(x / scale)).
 *
 * vibe_fp8_quantize_rows: X bf16 [R,d] -> Xq e4m3 [R,d] (uint8 codes), row_scale f32 [R].   d % 8 == 0.
 * vibe_fp8_pack_weights : W bf16 [E_loc,K,N] (the layout of W1/W3/W2) -> Wq e4m3 [E_loc,N,K] (K contiguous)
 *                         and scale f32 [E_loc]; a one-time pass (weights are static in serving).
 * vibe_grouped_ffn_fp8  : per resident expert e and row r of its segment
 *        g = sx[r] s1[e] (xq . w1q),  u = sx[r] s3[e] (xq . w3q),  h = silu(g) u,
 *        Hq[r,:] = e4m3(h / h_scale[e]),   Y[r,:] = bf16( h_scale[e] s2[e] (hq . w2q) )
 *   e4m3 x e4m3 products accumulated in fp32 on the tensor cores (tcgen05 kind::f8f6f4).
 *   Xq [R_cap,d], Hq_ws [R_cap,f] e4m3; W1q,W3q [E_loc,f,d], W2q [E_loc,d,f] e4m3; Y [R_cap,d] bf16;
 *   row_scale [R_cap], s1,s3,s2,h_scale [E_loc] f32 (h_scale: a STATIC, caller-chosen scale of the
 *   intermediate, e.g. a calibrated absmax / 448).  d % 128 == 0, f % 128 == 0.  All device pointers,
 *   asynchronous on `stream`, same offsets / ownership / error conventions as vibe_grouped_ffn.
 * ---------------------------------------------------------------------------------- */
VIBE_API vibe_status vibe_fp8_quantize_rows(const void* X, int32_t R, int32_t d, void* Xq, float* row_scale,
                                            void* stream);
VIBE_API vibe_status vibe_fp8_pack_weights(const void* W, int32_t E_loc, int32_t K, int32_t N, void* Wq,
                                           float* scale, void* stream);
VIBE_API vibe_status vibe_grouped_ffn_fp8(const void* Xq, const float* row_scale, const int32_t* offsets,
                                          int32_t E_loc, int32_t R_cap, int32_t d, int32_t f, const void* W1q,
                                          const float* s1, const void* W3q, const float* s3, const void* W2q,
                                          const float* s2, const float* h_scale, void* Hq_ws, void* Y,
                                          void* stream);

/* ------------------------------------------------------------------------------------
 * f2 as SURVEY 8(f) words it: "e4m3, BLOCK-SCALED".  The same FFN with one power-of-two (UE8M0) scale per
 * operand row and 32 elements of the contraction dimension K, applied by the tensor core itself
 * (tcgen05.mma kind::mxf8f6f4.block_scale).  The paper says only "Precision: FP8" (Table 2a);
 * the recipe is DESIGN.md readings Q5-Q8:
 *   block  = `block` (32 | 128) consecutive K elements of a row (a token row of X / H, one output feature of a
 *            weight matrix); 128 = the same scale stored for its four 32-blocks;
 *   scale  = 2^e, e = the smallest integer with amax <= 448 * 2^e, clamped to [-127, 127], 0 for an all-zero
 *            block; stored as the byte e + 127, ONE BYTE PER 32 ELEMENTS;   code = e4m3_rne(x / 2^e)  (exact division).
 * Scale-factor layouts (byte offset of the scale of row r -- a token row, or output feature n -- and 32-block b;
 * KS = K/128):
 *   VIBE_MX_SF_ROWMAJOR  [rows][K/32]:                 r * (K/32) + b
 *   VIBE_MX_SF_TOKENS    [KS][32][Rb] 32-bit words:    (((b/4)*32 + r%32) * Rb + r/32) * 4 + b%4,
 *                        Rb = ceil(R_cap/32) rounded up to a multiple of 4   (what vibe_grouped_ffn_mxfp8 reads:
 *                        an aligned {4 row blocks x 32 rows} box of it is the tensor core's scale layout, and a tile
 *                        may start at its row block 0 or 2, i.e. on any multiple of 64 rows)
 *   VIBE_MX_SF_GATE_UP   [E_loc][KS][N/64] chunks of 512 B, W1 and W3 JOINTLY (the gate|up kernel keeps 64 features
 *                        of each in one CTA):  ((e*KS + b/4)*(N/64) + n/64)*512 + (n%32)*16 + ((n%64)/32 + 2*up)*4 + b%4
 *   VIBE_MX_SF_DOWN      [E_loc][KS][N/128] chunks:    ((e*KS + b/4)*(N/128) + n/128)*512 + (n%32)*16 + ((n%128)/32)*4 + b%4
 * vibe_mxfp8_sf_bytes(which, rows, K, E_loc): bytes of such an array (rows = R / R_cap / N).
 *
 * vibe_mxfp8_quantize_rows: X bf16 [R,d] -> Xq e4m3 [R,d] + scales in ROWMAJOR or TOKENS layout (R_cap: row
 *                           capacity that fixes Rb; ignored for ROWMAJOR).  d % 128 == 0.
 * vibe_mxfp8_pack_weights : W bf16 [E_loc,K,N] -> Wq e4m3 [E_loc,N,K] + scales; role DOWN writes a DOWN array,
 *                           roles GATE and UP write their halves of ONE GATE_UP array (call once with W1 / GATE
 *                           and once with W3 / UP on the same `sf`).  K, N % 128 == 0.  One-time pass.
 * vibe_grouped_ffn_mxfp8  : per resident expert and row:  g = x . w1, u = x . w3 on the block-dequantised values
 *                           (fp32 accumulate), h = silu(g) u, (Hq, Hsf) = block-32 quantisation of h along f,
 *                           Y = bf16(deq(hq) . w2).  Xq [R_cap,d], Xsf TOKENS layout (K = d); Hq_ws [R_cap,f] and
 *                           Hsf_ws (TOKENS layout, K = f) are scratch; `offsets` MUST be multiples of 64
 *                           (vibe_permute with align = 64): token tiles start on an even scale row block.
 *                           d % 128 == 0, f % 128 == 0.  Conventions as vibe_grouped_ffn.
 * ---------------------------------------------------------------------------------- */
enum { VIBE_MX_SF_ROWMAJOR = 0, VIBE_MX_SF_TOKENS = 1, VIBE_MX_SF_GATE_UP = 2, VIBE_MX_SF_DOWN = 3 };
enum { VIBE_MX_ROLE_DOWN = 0, VIBE_MX_ROLE_GATE = 1, VIBE_MX_ROLE_UP = 2 };
VIBE_API size_t vibe_mxfp8_sf_bytes(int32_t which, int32_t rows, int32_t K, int32_t E_loc);
VIBE_API vibe_status vibe_mxfp8_quantize_rows(const void* X, int32_t R, int32_t d, int32_t block, void* Xq, void* sf,
                                              int32_t sf_layout, int32_t R_cap, void* stream);
VIBE_API vibe_status vibe_mxfp8_pack_weights(const void* W, int32_t E_loc, int32_t K, int32_t N, int32_t block,
                                             int32_t role, void* Wq, void* sf, void* stream);
VIBE_API vibe_status vibe_grouped_ffn_mxfp8(const void* Xq, const void* Xsf, const int32_t* offsets, int32_t E_loc,
                                            int32_t R_cap, int32_t d, int32_t f, const void* W1q, const void* W3q,
                                            const void* sf13, const void* W2q, const void* sf2, void* Hq_ws,
                                            void* Hsf_ws, void* Y, void* stream);

/* ------------------------------------------------------------------------------------
 * a6.  Per-expert latency profile: measured vibe_grouped_ffn time versus tokens per
 * expert, at warmed steady state -- "Each GPU is warmed to steady-state operating
 * conditions and profiled independently using the fused MoE kernel across a range of
 * token counts.  This produces a function f_g(n)" (protocol P:L335, L420).
 * Readings M1-M4.
 *
 *   mode 0 (uniform): every one of the E_loc experts receives n = tokens_per_expert[p]
 *           rows; latency_us[p] = median kernel time / E_loc   (per-expert cost l(n))
 *   mode 1 (solo):    expert 0 receives n rows, the others none; latency_us[p] = median time
 * Times are CUDA-event times of `iters` back-to-back executions (each timed separately)
 * after max(warmup, 1) untimed calls per point.  The timed executions replay one call
 * captured into a CUDA graph, on a stream of the sweep's own, so that an event pair
 * brackets the kernels and not the host's work between launches (a lone small expert
 * takes less device time than the host needs to launch it).  Every timed execution starts
 * COLD: before its first event an evict_last read sweep over 256 MB (twice the L2; a region at
 * the end of ws) evicts what the previous execution left in L2 -- a sweep point whose weights
 * fit the 126 MB L2 would otherwise be replayed on L2-resident weights and read faster than it
 * does inside a model.  Activations are an arbitrary
 * finite pattern written by the library into ws (latency does not depend on values).
 * This call SYNCHRONISES the stream (before the sweep) and returns when the sweep is done.  tokens_per_expert, latency_us, samples_us: HOST.
 * samples_us: optional host [n_points*iters] per-iteration times (NULL to skip).
 * ws: vibe_workspace_bytes(VIBE_WS_PROFILE, T = max tokens_per_expert, ...) bytes.
 * ---------------------------------------------------------------------------------- */
VIBE_API vibe_status vibe_profile_expert_latency(int32_t E_loc, int32_t d, int32_t f, const void* W1,
                                                 const void* W3, const void* W2,
                                                 const int32_t* tokens_per_expert /*host*/, int32_t n_points,
                                                 int32_t mode, int32_t warmup, int32_t iters,
                                                 float* latency_us /*host*/, float* samples_us /*host|NULL*/,
                                                 void* ws, size_t ws_bytes, void* stream);

/* Measurement utility (the protocol of a6, for callers that time kernels themselves): reads `bytes` of `scratch`
 * (device, 16-byte aligned; use >= 2 x the L2 size, 256 MB on B200) with the L2 evict_last policy, which evicts
 * what earlier kernels left in L2 -- including the evict_last operand lines of the FFN kernels that a plain memset
 * would not displace.  Asynchronous on `stream`; the buffer's contents are not changed. */
VIBE_API vibe_status vibe_l2_flush(void* scratch, size_t bytes, void* stream);

/* a6 in the paper's precision (f2): the same profile of vibe_grouped_ffn_fp8 (packed weights and scales as there).
 * ws: vibe_workspace_bytes(VIBE_WS_PROFILE, T = max tokens_per_expert, ...) rounded up to 256, plus
 * 4 * E_loc * max(tokens_per_expert) rounded up to 256 bytes. */
VIBE_API vibe_status vibe_profile_expert_latency_fp8(int32_t E_loc, int32_t d, int32_t f, const void* W1q,
                                                     const float* s1, const void* W3q, const float* s3,
                                                     const void* W2q, const float* s2, const float* h_scale,
                                                     const int32_t* tokens_per_expert /*host*/, int32_t n_points,
                                                     int32_t mode, int32_t warmup, int32_t iters,
                                                     float* latency_us /*host*/, float* samples_us /*host|NULL*/,
                                                     void* ws, size_t ws_bytes, void* stream);

/* a6 for the BLOCK-SCALED FP8 FFN (packed weights / scales as vibe_grouped_ffn_mxfp8).  Segments start on multiples of
 * 64 rows and are roundup(n, 64) rows long -- what vibe_permute with align = 64 hands that kernel -- so l(n) is a step
 * function of n with steps of 64.  ws: with n' = max(roundup(max tokens_per_expert, 64), 64) and R' = E_loc * n':
 * vibe_workspace_bytes(VIBE_WS_PROFILE, T = n', ...) rounded up to 256, plus vibe_mxfp8_sf_bytes(TOKENS, R', d) and
 * vibe_mxfp8_sf_bytes(TOKENS, R', f), each rounded up to 256 bytes. */
VIBE_API vibe_status vibe_profile_expert_latency_mxfp8(int32_t E_loc, int32_t d, int32_t f, const void* W1q,
                                                       const void* W3q, const void* sf13, const void* W2q,
                                                       const void* sf2, const int32_t* tokens_per_expert /*host*/,
                                                       int32_t n_points, int32_t mode, int32_t warmup, int32_t iters,
                                                       float* latency_us /*host*/, float* samples_us /*host|NULL*/,
                                                       void* ws, size_t ws_bytes, void* stream);


/* ------------------------------------------------------------------------------------
 * The whole layer (a1..a5) as one call: enqueues route -> permute -> grouped FFN ->
 * combine on `stream` using one caller-provided device arena.
 * arena: vibe_workspace_bytes(VIBE_WS_LAYER, ...) bytes, 256-byte aligned.
 * Outputs: out [T,d] bf16, counts [E] i32 (device).  Optional device outputs topk_ids /
 * topk_w may be NULL (then they live in the arena).
 * ---------------------------------------------------------------------------------- */
VIBE_API vibe_status vibe_moe_layer_forward(const vibe_route_cfg* cfg /*host*/, const float* logits,
                                            const void* X, const int32_t* expert_map, int32_t T, int32_t d,
                                            int32_t f, int32_t E_loc, const void* W1, const void* W3,
                                            const void* W2, void* out, int32_t* counts, int32_t* topk_ids,
                                            float* topk_w, void* arena, size_t arena_bytes, void* stream);

/* Same, end to end from HOST buffers: copies logits_h and X_h (pinned or pageable host
 * memory) to the device, runs the layer, copies out_h and counts_h back, and waits for
 * the stream.  Weights, select_bias and expert_map stay device-resident (model state).
 * arena additionally holds the device copies: vibe_workspace_bytes(VIBE_WS_LAYER_HOST, ...).
 * The tokens are cut into chunks (a token's output does not depend on the other tokens of
 * the batch; the histograms of the chunks are summed on the device): chunk c's copy-in,
 * layer and copy-out run on three streams (two library-owned copy streams, created on
 * first use, ordered after the work already on `stream`), so that with PINNED host
 * buffers the PCIe transfers of both directions overlap the kernels.  The chunk count
 * is chosen from the shapes by a pipeline estimate. */
VIBE_API vibe_status vibe_moe_layer_forward_host(const vibe_route_cfg* cfg /*host*/,
                                                 const float* logits_h /*host*/, const void* X_h /*host*/,
                                                 const int32_t* expert_map, int32_t T, int32_t d, int32_t f,
                                                 int32_t E_loc, const void* W1, const void* W3, const void* W2,
                                                 void* out_h /*host*/, int32_t* counts_h /*host*/, void* arena,
                                                 size_t arena_bytes, void* stream);

/* vibe_moe_layer_forward_host with the number of token chunks given: n_chunks = 0 lets the
 * library choose, 1 is the unpipelined path, at most 8.  Chunks hold a multiple of 16
 * tokens (the last one the remainder); out_h and counts_h do not depend on n_chunks. */
VIBE_API vibe_status vibe_moe_layer_forward_host_chunked(const vibe_route_cfg* cfg /*host*/,
                                                         const float* logits_h /*host*/, const void* X_h /*host*/,
                                                         const int32_t* expert_map, int32_t T, int32_t d,
                                                         int32_t f, int32_t E_loc, const void* W1, const void* W3,
                                                         const void* W2, void* out_h /*host*/,
                                                         int32_t* counts_h /*host*/, int32_t n_chunks, void* arena,
                                                         size_t arena_bytes, void* stream);

/* ASYNCHRONOUS host entry: the same work as vibe_moe_layer_forward_host with one token chunk, but the call only
 * ENQUEUES it -- copy-in on the library's copy-in stream, the layer on `stream`, copy-out on the library's copy-out
 * stream -- and returns a ticket; vibe_host_wait(ticket) blocks until out_h and counts_h of that call are filled.
 * Issued back to back with TWO arenas (and two result buffers), step i+1's copy-in and step i-1's copy-out overlap
 * step i's kernels, and every step still streams the weights once over the whole batch (no token chunks).
 * Contract: host buffers must be PINNED (pageable memory makes the copies synchronous: still correct, no overlap);
 * an arena, its out_h / counts_h and the host inputs of a call belong to that call until its ticket has been waited
 * for; at most 8 tickets may be outstanding per device; tickets are waited for in any order, each exactly once.
 * out_h / counts_h are bit-identical to vibe_moe_layer_forward_host's. */
VIBE_API vibe_status vibe_moe_layer_forward_host_async(const vibe_route_cfg* cfg /*host*/,
                                                       const float* logits_h /*host*/, const void* X_h /*host*/,
                                                       const int32_t* expert_map, int32_t T, int32_t d, int32_t f,
                                                       int32_t E_loc, const void* W1, const void* W3, const void* W2,
                                                       void* out_h /*host*/, int32_t* counts_h /*host*/, void* arena,
                                                       size_t arena_bytes, void* stream, int32_t* ticket /*host, out*/);
VIBE_API vibe_status vibe_host_wait(int32_t ticket);

/* The whole layer with the FP8 FFN (f2): route -> e4m3 quantisation of the token rows (on an expert-parallel
 * shard only of the tokens that have a resident expert) -> permute (one-byte rows) -> row-scale gather -> vibe_grouped_ffn_fp8 -> combine.  Packed weights / scales as in
 * vibe_grouped_ffn_fp8; arena: vibe_workspace_bytes(VIBE_WS_LAYER_FP8, ...) bytes, 256-byte aligned.
 * out [T,d] bf16, counts [E] i32 (device).  d % 128 == 0, f % 128 == 0. */
VIBE_API vibe_status vibe_moe_layer_forward_fp8(const vibe_route_cfg* cfg /*host*/, const float* logits,
                                                const void* X, const int32_t* expert_map, int32_t T, int32_t d,
                                                int32_t f, int32_t E_loc, const void* W1q, const float* s1,
                                                const void* W3q, const float* s3, const void* W2q, const float* s2,
                                                const float* h_scale, void* out, int32_t* counts, void* arena,
                                                size_t arena_bytes, void* stream);

/* The whole layer with the BLOCK-SCALED FP8 FFN: route -> block-32 quantisation of the token rows (ROWMAJOR scales;
 * on an expert-parallel shard only tokens with a resident expert) -> permute with align = 64 (one-byte rows) ->
 * scale gather into the TOKENS layout -> vibe_grouped_ffn_mxfp8 -> combine.  Weights / scales as there;
 * arena: vibe_workspace_bytes(VIBE_WS_LAYER_MXFP8, ...) bytes, 256-byte aligned.  d % 128 == 0, f % 128 == 0. */
VIBE_API vibe_status vibe_moe_layer_forward_mxfp8(const vibe_route_cfg* cfg /*host*/, const float* logits,
                                                  const void* X, const int32_t* expert_map, int32_t T, int32_t d,
                                                  int32_t f, int32_t E_loc, const void* W1q, const void* W3q,
                                                  const void* sf13, const void* W2q, const void* sf2, void* out,
                                                  int32_t* counts, void* arena, size_t arena_bytes, void* stream);

/* Workspace sizing.  `which` selects the consumer. */
enum {
  VIBE_WS_PERMUTE = 0,
  VIBE_WS_FFN = 1,
  VIBE_WS_PROFILE = 2, /* T = max tokens per expert of the sweep */
  VIBE_WS_LAYER = 3,
  VIBE_WS_LAYER_HOST = 4,
  VIBE_WS_LAYER_FP8 = 5,
  VIBE_WS_LAYER_MXFP8 = 6
};
VIBE_API size_t vibe_workspace_bytes(int32_t which, int32_t T, int32_t k, int32_t E, int32_t E_loc, int32_t d,
                                     int32_t f, int32_t align);
/* Upper bound on offsets[E_loc]: min(T*k, T*E_loc) + E_loc*(align-1). */
VIBE_API int64_t vibe_rows_cap(int32_t T, int32_t k, int32_t E_loc, int32_t align);

VIBE_API const char* vibe_status_string(vibe_status s);
VIBE_API const char* vibe_last_error(void); /* thread-local, never NULL */
VIBE_API int32_t vibe_version(void);
/* Number of kernel launches this library has issued on this thread since load
 * (memsets and copies not counted): lets a caller report how many of ITS kernels ran. */
VIBE_API int64_t vibe_launch_count(void);

/* ====================================================================================
 * Host-side placement (fp64, no device work).  P:L182-L196, Algorithm 1 Phase 2.
 * ==================================================================================== */

/* Latency model (reading M1): monotone piecewise-linear per-expert latency l(n) through
 * (0,0) and the profiled points (running max applied), linear extrapolation with the last
 * segment's slope.  E_prof: experts resident when profiled in uniform mode, so the
 * whole-kernel latency with n tokens in total is F(n) = E_prof * l(n / E_prof).
 * tokens must be strictly increasing and > 0.  NULL model pointer means f(n) = n. */
typedef struct {
  int32_t n_points;
  const double* tokens;     /* host [n_points] */
  const double* latency_us; /* host [n_points] */
  int32_t E_prof;
} vibe_latency_model;

enum { VIBE_MODEL_A = 0, /* paper-faithful scalar model  L_g = F(sum_e load_e) */
       VIBE_MODEL_B = 1  /* per-expert profile           L_g = sum_e l(load_e)   (L4)     */ };

/* a7.  score(S) = max_g L_g / scale[g]   -- "T = max_g f_g(n_g)", n_g = sum_{e in S_g} w_e
 * with f_g = f / sigma_g (M5).  assign [E] in [0,G); load [E] tokens;
 * scale [G] in (0,1]; per_bin [G] or NULL receives L_g / scale[g].
 * Returns the score, or a negative value on invalid arguments (see vibe_last_error). */
VIBE_API double vibe_placement_eval(const int32_t* assign, const double* load, int32_t E, int32_t G,
                                    const double* scale, const vibe_latency_model* m, int32_t model_kind,
                                    double* per_bin);

/* a8.  ViBE's latency-aware greedy (Algorithm 1 Phase 2):
 *   N = sum_e load_e; s_g = 1/f_g(N/E); tau_g = N s_g / sum_h s_h; experts in descending
 *   load (ties -> lower e); each to argmax_g (tau_g - n_g) (ties -> lower g) among bins
 *   with fewer than `cap` experts (cap = 0: unlimited; P:L260 uses cap = E/G). */
VIBE_API vibe_status vibe_placement_greedy(const double* load, int32_t E, int32_t G, const double* scale,
                                           const vibe_latency_model* m, int32_t cap, int32_t* assign);
/* Token-balanced baseline: "EPLB implicitly assumes f_g(n) = n" = the same greedy
 * with all scales equal (L3). */
VIBE_API vibe_status vibe_placement_token_balanced(const double* load, int32_t E, int32_t G, int32_t cap,
                                                   int32_t* assign);
/* vLLM's contiguous default: e -> floor(e*G/E). */
VIBE_API vibe_status vibe_placement_contiguous(int32_t E, int32_t G, int32_t* assign);

/* ====================================================================================
 * f1.  Online recalibration (host, fp64): drift detector and incremental placement update.
 * ==================================================================================== */

/* d = 1 - (w . w_ref) / (|w| |w_ref|)  -- the cosine distance between the current window
 * average and the reference load vector of one layer.  A zero vector gives 0
 * (reading D1).  Returns a negative value on invalid arguments. */
VIBE_API double vibe_drift_cosine(const double* w, const double* w_ref, int32_t E);

/* Algorithm 1 phase 3 bookkeeping (reading D3) for L layers x E
 * experts: a sliding window of the last `window` per-pass load vectors (paper: 100); every
 * H-th pass (paper: 10), if a reference exists and no cooldown is running, the per-layer
 * distances between the window mean and the reference are computed; recalibration is
 * triggered when any exceeds delta (paper: 0.05).  The library owns the monitor object
 * (create / destroy); all arrays are HOST, row-major [L,E]. */
typedef struct vibe_drift_monitor vibe_drift_monitor;
VIBE_API vibe_drift_monitor* vibe_drift_monitor_create(int32_t L, int32_t E, int32_t window, int32_t H,
                                                       double delta); /* NULL on error */
VIBE_API void vibe_drift_monitor_destroy(vibe_drift_monitor* m);
/* "Snapshot w_ref <- current load vectors": explicit reference, e.g. the profiling W. */
VIBE_API vibe_status vibe_drift_monitor_set_reference(vibe_drift_monitor* m, const double* W);
/* One forward pass.  Returns 1 if recalibration is triggered on this pass, 0 if not, -1 on
 * error.  *checked (optional) = 1 when distances were computed on this pass, and then
 * d_out[L] (optional) holds them. */
VIBE_API int32_t vibe_drift_monitor_push(vibe_drift_monitor* m, const double* loads, double* d_out,
                                         int32_t* checked);
/* After a rearrangement: "w_ref <- w for all l; cooldown for H forward passes". */
VIBE_API vibe_status vibe_drift_monitor_rearranged(vibe_drift_monitor* m);
VIBE_API vibe_status vibe_drift_monitor_window_mean(const vibe_drift_monitor* m, double* W);

/* Algorithm 2 (prose P:L210-L214, L426-L428), one layer, in place on assign[E]:
 *   repeat  g+ = slowest bin, g- = fastest bin (ties -> lower g);
 *           stop if max_g L_g <= (1+eps) * mean_g L_g;
 *           over all (e_i in g+, e_j in g-) take the swap with the largest reduction of
 *           max(L_g+, L_g-) (reading D2; ties -> lowest (e_i, e_j)); stop if none reduces it;
 *           apply the swap;
 *   until max_swaps swaps were applied.
 * L_g as in vibe_placement_eval (model kind A or B, scale = sigma_g).  Per-bin expert counts
 * are preserved.  n_swaps (optional) receives the number applied; swaps (optional, capacity
 * 2*max_swaps) the pairs (e_i, e_j) in order. */
VIBE_API vibe_status vibe_placement_swap_refine(int32_t* assign, const double* load, int32_t E, int32_t G,
                                                const double* scale, const vibe_latency_model* m,
                                                int32_t model_kind, double eps, int32_t max_swaps,
                                                int32_t* n_swaps, int32_t* swaps);

#ifdef __cplusplus
}
#endif
#endif /* VIBE_H_ */
