// ffn.cu -- a4: grouped SwiGLU expert FFN (vibe_grouped_ffn) on 5th-gen tensor cores.
//
// Two launches of one persistent, warp-specialised tcgen05 kernel; the grid is 74 CTA PAIRS
// (clusters of 2, one CTA per SM) and every MMA is a cta_group::2 instruction of M = 256.
//
// "Swap-AB": the WEIGHTS are the UMMA A operand (M side = output features, always full
// tiles) and the TOKENS are the B operand (N side).  The ragged dimension -- rows per expert --
// therefore lands on UMMA N, which is a runtime field of the instruction descriptor with a
// granularity of 16: an expert with n rows costs roundup(n,16) columns of MMA work, not
// roundup(n,128) rows, and the last tile of every expert is exactly as wide as it needs to be.
//
//   GEMM-1  H^T[n, r] = silu(W1[s]^T Xp^T) * (W3[s]^T Xp^T)      K = d
//           pair tile = 128 features x <=256 tokens.  Each CTA's A tile is two 64-feature
//           TMA atoms: its 64 gate features (W1) in TMEM lanes 0..63 and the SAME 64 features
//           of W3 in lanes 64..127, so ONE MMA stream produces gate and up; the epilogue
//           warps of the two lane halves swap 32-column blocks through shared memory and
//           apply SwiGLU out of TMEM (H never exists in fp32 in HBM).
//   GEMM-2  Y^T[n, r] = W2[s]^T H^T                               K = f
//           pair tile = 256 features x <=256 tokens.
// Operands:
//   A (weights [E_loc,K,N], N contiguous = "MN-major"): ONE 3-D TMA map (N, K, E_loc), 64x64
//       boxes, consumed IN PLACE through MN-major UMMA descriptors -- no weight repacking.
//   B (activations [R_cap,K], K-major): ONE 2-D TMA map over all permuted rows; the row
//       coordinate comes from the device-side offsets -> no per-expert descriptors, no host
//       sync.  Each CTA of the pair loads HALF of the token tile (cta_group::2 takes N/2
//       columns of B from each CTA), so per-SM shared-memory fill is 32 KB per 64-deep K step.
// Token columns past the end of the expert's segment are computed on whatever the box holds
// and masked at the store (columns are independent, nothing leaks); rows past R_cap are
// zero-filled by TMA.
// Pipeline: warp 0 = TMA producer (both CTAs), warp 1 = UMMA issuer (leader CTA) + TMEM owner,
// warps 2.. = epilogue (4 for GEMM-1, 8 for GEMM-2).  Producer and issuer are warp-uniform loops
// with elect.sync around the instructions (operands stay in uniform registers).  6 smem stages
// x 32 KB, 2 TMEM accumulator stages x 256 columns so the epilogue of tile i overlaps the MMAs
// of tile i+1.
// Tiles: an expert's rows are cut into EQUAL token tiles (multiples of 16, <= 256); tile order is
// expert-major, then feature block, then token tile fastest, handed to the pairs round by round
// with a rotation (tile_of), so pairs that run at the same time share a weight tile through L2
// (both operands evict_last), run K steps of equal length, and each weight byte leaves HBM once.
// Epilogue: tcgen05.ld 32 lanes x 32 columns, bf16x2 pack + one shuffle + byte permute per token
// pair (the output is the TRANSPOSE of the accumulator), 4-byte stores of two adjacent features.
//
// Split-K (S8(f) f4, the few-active-experts regime): when the launch has at most half as many tiles as the grid has
// CTA pairs (a lone expert of a decode step: 16 / 28 tiles for 74 pairs, each pair limited to ~140 GB/s of weight
// streaming), every tile's K range is cut into S = min(pairs / tiles, 8, K steps / 4) slices, one (tile, slice) unit
// per pair.  A unit dumps its fp32 accumulator to the caller's workspace; the LAST unit of a tile portion to
// arrive (one counter per tile, CTA rank and epilogue warp role) sums the S partials in slice order -- a fixed
// order, so the result does not depend on which unit came last -- and runs the normal epilogue on the sum.
// S is derived on the device from `offsets`, like everything else.
//
// ONE kernel, three operand kinds (template parameter kKind) -- producer, MMA issuer, tile scheduler, split-K and
// the epilogue skeleton are shared; a kind changes only what is listed here:
//   KIND_BF16  bf16 x bf16 (kind::f16), K = 16 per MMA, 64 K elements per 128-byte smem row; the weights are consumed in
//              place, [E_loc,K,N] N-contiguous: MN-major A descriptors, TMA coordinates (n, k, e)
//   KIND_F8    e4m3 x e4m3 (kind::f8f6f4), K = 32 per MMA, 128 K elements per row; weights pre-quantised and
//              pre-transposed to [E_loc,N,K] (vibe_fp8_pack_weights): K-major A, TMA coordinates (k, n, e); per-row,
//              per-expert and static H scales multiply the accumulators in the epilogue; GEMM-1 writes H as e4m3
//              (readings Q1-Q4)
//   KIND_MXF8  e4m3 BLOCK-SCALED (kind::mxf8f6f4.block_scale; readings Q5-Q8): one UE8M0 scale per operand row and 32
//              K elements, applied by the tensor core.  The scales of a K = 128 stage travel with the stage (weights:
//              one 512-byte chunk already in TMEM order; tokens: aligned {4 row blocks x 32 rows} boxes of the
//              [K/128][32][Rb] word array, which land in TMEM order; a tile that starts on a 64-row boundary reads
//              them from column 0 or 2 of its chunk), are copied to TMEM by tcgen05.cp ahead of the stage's four MMAs
//              (same issuing thread: ordered with them), and the instruction descriptor's scale-factor ids pick the
//              K-block's byte.  Token tiles are multiples of 64 rows and at most 192 (2 x 192 accumulator columns + 12
//              scale columns fit the 512 TMEM columns); no scale arithmetic is left in the epilogues; GEMM-1
//              block-quantises H per row and 32 features (one warp = one block: redux.sync max).
//
// Semantics: include/vibe.h (vibe_grouped_ffn, vibe_grouped_ffn_fp8, vibe_grouped_ffn_mxfp8); F1-F4, Q1-Q8.
#include <mutex>
#include <unordered_map>
#include <string>
#include <cstring>

#include "common.cuh"
#include "ptx.cuh"

namespace vibe {
namespace {

enum { KIND_BF16 = 0, KIND_F8 = 1, KIND_MXF8 = 2 };
__host__ __device__ constexpr int bk_of(int kind) { return kind == KIND_BF16 ? 64 : 128; }      // K elements per smem stage (128 bytes)
__host__ __device__ constexpr int umma_k_of(int kind) { return kind == KIND_BF16 ? 16 : 32; }  // K per MMA instruction (32 bytes)
__host__ __device__ constexpr int tn_of(int kind) { return kind == KIND_MXF8 ? 192 : 256; }    // tokens per tile = TMEM columns per accumulator
__host__ __device__ constexpr int talign_of(int kind) { return kind == KIND_MXF8 ? 64 : 16; }  // token tiles are multiples of this

constexpr int TN = 256;                 // largest token tile = max UMMA N
constexpr int STAGES = 6;
constexpr int ATOM_BYTES = 64 * 128;            // 8 KB : 64 features x 128 bytes of K (or 64 K-rows x 128 bytes of features), SW128
constexpr int A_BYTES = 2 * ATOM_BYTES;         // 16 KB: this CTA's 128 accumulator lanes
constexpr int B_BYTES = (TN / 2) * 128;         // 16 KB: this CTA's half of the token tile
constexpr int STAGE_BYTES = A_BYTES + B_BYTES;  // 32 KB
constexpr int NARROW_ROWS = 32;                 // rows of the small activation box (per CTA)
constexpr int XCHG_BYTES = 16384;               // gate/up swap: 2 warp pairs x 2 directions x 4 KB
constexpr int SX_BYTES = 4 * TN * 4;            // KIND_F8 GEMM-1: the tile's row scales, one 1 KB slice per epilogue warp
// block-scaled kind: per-CTA activation bytes of a stage, and where the stage keeps its scale factors
constexpr int B_BYTES_MX = (tn_of(KIND_MXF8) / 2) * 128;   // 12 KB
constexpr int SFA_OFF = A_BYTES + B_BYTES_MX;   // 512 B : this CTA's 128 weight rows x 4 K-blocks
constexpr int SFB_OFF = SFA_OFF + 512;          // 1 KB  : up to two 128-row chunks of token scales x 4 K-blocks
static_assert(SFB_OFF + 1024 <= STAGE_BYTES, "scale factors must fit behind the narrower activation tile");
constexpr uint32_t SF_TMEM_COL = 2 * tn_of(KIND_MXF8);     // columns 384.. : SFA (4) then SFB (8)
// warps: 0 = TMA producer, 1 = MMA issuer, 2.. = epilogue.  GEMM-1 has 4 epilogue warps (its SwiGLU
// epilogue needs ~200 registers per thread); the down projection has 8 -- two per TMEM lane quarter,
// alternating 32-column blocks -- because with a short K loop (f = 768: 12 K steps per tile) one warp
// per quarter could not drain a 256-column accumulator as fast as the tensor pipe fills the next
// (ncu at the C2 shape: tensor pipe 33 % active with 4 warps).
__host__ __device__ constexpr int num_threads(int mode) { return mode == 0 ? 192 : 320; }
constexpr int MAX_SLOTS = 512;
constexpr int TMEM_COLS = 512;
// split-K workspace: partial accumulators [unit][column][256 features of the pair tile] fp32, then the counters
constexpr int SPLIT_MAX = 8;               // K slices per tile at most
constexpr int SPLIT_MIN_STEPS = 4;         // K steps per slice at least
constexpr int SPLIT_MAX_UNITS = 128;       // >= CTA pairs of any supported device (B200: 74)
constexpr size_t SPLIT_PART_BYTES = (size_t)SPLIT_MAX_UNITS * TN * 256 * sizeof(float);
constexpr int SPLIT_COUNTERS = SPLIT_MAX_UNITS * 16;     // per tile: 2 CTA ranks x 8 epilogue-warp roles
constexpr int TILE_CTRS = 16;               // [0], [8]: the next-unit counters of GEMM-1 / GEMM-2 (dynamic tile scheduler)
constexpr size_t SPLIT_CNT_BYTES = (2 * (size_t)SPLIT_COUNTERS + TILE_CTRS) * sizeof(int);       // zeroed per call
constexpr size_t SPLIT_WS_BYTES = SPLIT_PART_BYTES + SPLIT_CNT_BYTES;   // partials | counters of GEMM-1 | of GEMM-2 | unit counters
constexpr int RING = 4;                     // unit ids in flight between the fetching warp and the other roles of a pair

// what the e4m3 kinds need beyond the bf16 kernel's arguments
struct FfnAux {
  CUtensorMap tmSFB;          // KIND_MXF8 token scales : u32 [K/128][32][Rb]
  CUtensorMap tmSFW;          // KIND_MXF8 weight scales: u32 [chunks][128 words], one 512-byte chunk per (expert, K stage, CTA feature tile)
  const float* row_scale;     // KIND_F8 GEMM-1: sx [R_cap]
  const float* sw0;           // KIND_F8: per-expert weight scale (W1 | W2)
  const float* sw1;           // KIND_F8 GEMM-1: W3's
  const float* h_scale;       // KIND_F8: static per-expert scale of H
  uint8_t* hsf;               // KIND_MXF8 GEMM-1: scales of H, written in the token-scale layout (K = f)
  int Rb;                     // KIND_MXF8: words per (K stage, lane) row of the token-scale arrays
  int wchunks;                // KIND_MXF8: weight chunks per (expert, K stage)
};

struct SmemTail {
  uint64_t full[STAGES];          // leader CTA: both CTAs' TMA bytes of a stage have landed
  uint64_t empty[STAGES];         // each CTA: the MMAs reading the stage have retired
  uint64_t tfull[2];              // each CTA: accumulator stage complete
  uint64_t tempty[2];             // leader CTA: all 8 epilogue warps of the pair drained it
  uint64_t rfull[RING];           // each CTA: ring slot holds the next unit id of the pair
  uint64_t rempty[RING];          // leader CTA: every consuming warp of the pair has read the slot
  int32_t ring[RING];             // unit ids (-1: no more work), written by the leader's producer warp in BOTH CTAs
  uint32_t tmem_base;
  int32_t total_t_tiles;
  int32_t split;                  // K slices of a split tile (1 = no split-K)
  int32_t split_from;             // first split tile: tiles [split_from, total) are cut into `split` K slices
  int32_t off[MAX_SLOTS + 1];     // segment starts (rows)
  int32_t cum[MAX_SLOTS + 1];     // exclusive prefix of token tiles per slot
  int32_t tsz[MAX_SLOTS];         // rows per token tile of the slot (multiple of 16, <= TN)
};
constexpr size_t SMEM_BYTES = 1024 + (size_t)STAGES * STAGE_BYTES + XCHG_BYTES + SX_BYTES + sizeof(SmemTail);
static_assert(SMEM_BYTES <= 232448, "exceeds the 227 KB dynamic shared memory of sm_100");

struct TileCursor {
  int e = 0;
  // tile id -> (slot e, feature block, token tile).  Tile ids are monotone per CTA, so e only advances.
  __device__ __forceinline__ void decode(const SmemTail* t, int tile, int NB, int& f_blk, int& t_blk) {
    while (tile >= t->cum[e + 1] * NB) ++e;
    const int local = tile - t->cum[e] * NB;
    const int tt = t->cum[e + 1] - t->cum[e];
    f_blk = local / tt;
    t_blk = local - f_blk * tt;
  }
};

// Tile of CTA pair `pair` in round `rnd`: round r hands out tiles [r*P, (r+1)*P) ROTATED by r.
// Tile ids stay increasing per pair, every tile is taken exactly once, and a pair does not keep
// the same position inside a repeating cost pattern (with the plain stride P = 74, a layer whose
// experts all have a 256-row and a 128-row token tile gave half the pairs only the large tiles).
__device__ __forceinline__ int tile_of(int rnd, int pair, int P) { return rnd * P + (pair + rnd) % P; }

__device__ __forceinline__ uint32_t pack2_bf16(float lo, float hi) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&h);
}
__device__ __forceinline__ float swiglu(float g, float u) { return __fdividef(g, 1.0f + __expf(-g)) * u; }

// Store a 32-lane x 32-column block held one lane (= feature) per thread, v[i] = column
// (= token) i, into row-major out[token][feature].  Every lane first packs its OWN two tokens
// (i, i+1) of its feature into one bf16x2 word; lanes 2j / 2j+1 swap that word with one shuffle
// and a byte permute picks {token i: features f, f+1} in the even lane and {token i+1: f, f+1}
// in the odd lane -- per token pair: 1 cvt.bf16x2 + 1 shfl + 1 prmt + 1 store (the first version
// shuffled fp32 values and selected operands with SELs: 365 instructions per block against ~120
// now, and the down projection at K = 768 was bound by exactly this epilogue).
__device__ __forceinline__ void store_block_T(const float (&v)[32], __nv_bfloat16* __restrict__ out, size_t ld,
                                              int row0, int n_rows, int feat, bool feat_ok, int lane) {
  const int odd = lane & 1;
  const uint32_t sel = odd ? 0x3276u : 0x5410u;
  __nv_bfloat16* p = out + (size_t)(row0 + odd) * ld + (feat - odd);
  const size_t step = 2 * ld;
  if (n_rows >= 32) {
#pragma unroll
    for (int i = 0; i < 32; i += 2) {
      const uint32_t own = pack2_bf16(v[i], v[i + 1]);
      const uint32_t got = __shfl_xor_sync(0xffffffffu, own, 1);
      const uint32_t pk = __byte_perm(own, got, sel);
      if (feat_ok) *reinterpret_cast<uint32_t*>(p) = pk;
      p += step;
    }
  } else {
#pragma unroll
    for (int i = 0; i < 32; i += 2) {
      const uint32_t own = pack2_bf16(v[i], v[i + 1]);
      const uint32_t got = __shfl_xor_sync(0xffffffffu, own, 1);
      const uint32_t pk = __byte_perm(own, got, sel);
      if (feat_ok && i + odd < n_rows) *reinterpret_cast<uint32_t*>(p) = pk;
      p += step;
    }
  }
}

// The same block, gate-weighted and scattered: token i of the block goes to row asg[i] (its flat
// assignment index, assignment order) of `out`, scaled by that assignment's gate weight wt[i]; the
// product is rounded to bf16 once.  asg / wt of the tile's tokens sit in this warp's slice of shared
// memory (written before the accumulator was ready): broadcast LDS, no shuffles, no global latency.
__device__ __forceinline__ void store_block_T_scatter(const float (&v)[32], __nv_bfloat16* __restrict__ out,
                                                      size_t ld, int feat, bool feat_ok, int lane,
                                                      const float* __restrict__ wt, const int* __restrict__ asg) {
  const int odd = lane & 1;
  const uint32_t sel = odd ? 0x3276u : 0x5410u;
#pragma unroll
  for (int i = 0; i < 32; i += 2) {
    const float2 w = *reinterpret_cast<const float2*>(wt + i);
    const int dst = asg[i + odd];
    const uint32_t own = pack2_bf16(v[i] * w.x, v[i + 1] * w.y);
    const uint32_t got = __shfl_xor_sync(0xffffffffu, own, 1);
    const uint32_t pk = __byte_perm(own, got, sel);
    if (feat_ok && dst >= 0) *reinterpret_cast<uint32_t*>(out + (size_t)dst * ld + (feat - odd)) = pk;
  }
}

// The same transposed store for an e4m3 output (GEMM-1 writes Hq): every lane packs its own two tokens
// of its feature into an e4m3x2 halfword; one shuffle + byte permute give {token: features f, f+1}.
__device__ __forceinline__ void store_block_T_e4m3(const float (&v)[32], uint8_t* __restrict__ out, size_t ld, int row0,
                                                   int n_rows, int feat, bool feat_ok, int lane) {
  const int odd = lane & 1;
  const uint32_t sel = odd ? 0x0015u : 0x0040u;   // even: (own.b0, got.b0) = token i;  odd: (got.b1, own.b1) = token i+1
  uint8_t* p = out + (size_t)(row0 + odd) * ld + (feat - odd);
  const size_t step = 2 * ld;
#pragma unroll
  for (int i = 0; i < 32; i += 2) {
    const uint32_t own = ptx::pack2_e4m3(v[i], v[i + 1]);
    const uint32_t got = __shfl_xor_sync(0xffffffffu, own, 1);
    const uint32_t pk = __byte_perm(own, got, sel);
    if (feat_ok && i + odd < n_rows) *reinterpret_cast<uint16_t*>(p) = (uint16_t)pk;
    p += step;
  }
}


// ---- which unit a pair works on next --------------------------------------------------------------------------
// Static (no workspace): round r hands out units [r*P, (r+1)*P) rotated by r (tile_of).  Dynamic (workspace given):
// the pairs take the next unit from ONE global counter when they are ready for it, so that consecutive units -- the
// token tiles that share a weight tile -- are started within microseconds of each other by whichever pairs are free,
// and stay L2-resident for each other; under the static assignment the pairs drift apart by whole tiles over the
// rounds (tile costs differ with the ragged N) and every drifted sharer re-reads its weight tile from DRAM
// (profiles/: 1.5 x the algorithmic bytes).  Dynamic hand-out also balances the ragged tile costs.
// The leader CTA's producer warp fetches (one atomicAdd per unit, on demand: its latency hides behind the 6 stages
// the producer runs ahead) and publishes the id to a 4-slot ring in both CTAs; every other role of the pair reads it.
// A pair's FIRST unit is its own index in both schemes (no counter round trip in front of the first TMA: ~1 us of
// every launch, which is a tenth of a lone light expert's kernel); the counter hands out units num_pairs, ...
struct UnitCursor {
  int rnd = 0, idx = 0;
  uint32_t ph = 0;
  bool first = true;
};
__device__ __forceinline__ int next_unit_fetch(SmemTail* tail, unsigned int* ctr, int total, int pair, int num_pairs,
                                               UnitCursor& c, int lane) {
  if (ctr == nullptr) {
    const int u = tile_of(c.rnd, pair, num_pairs);
    ++c.rnd;
    return u < total ? u : -1;
  }
  if (c.first) {
    c.first = false;
    return pair < total ? pair : -1;
  }
  const int slot = c.idx;
  ptx::mbar_wait(ptx::smem_u32(&tail->rempty[slot]), c.ph ^ 1u);
  int u = 0;
  if (lane == 0) {
    u = (int)atomicAdd(ctr, 1u) + num_pairs;
    if (u >= total) u = -1;
    const uint32_t ra = ptx::smem_u32(&tail->ring[slot]), fa = ptx::smem_u32(&tail->rfull[slot]);
    ptx::st_shared_cluster_u32(ptx::mapa_u32(ra, 0), (uint32_t)u);
    ptx::st_shared_cluster_u32(ptx::mapa_u32(ra, 1), (uint32_t)u);
    ptx::mbar_arrive_release_cluster(ptx::mapa_u32(fa, 0));
    ptx::mbar_arrive_release_cluster(ptx::mapa_u32(fa, 1));
  }
  u = __shfl_sync(0xffffffffu, u, 0);
  if (++c.idx == RING) { c.idx = 0; c.ph ^= 1u; }
  return u;
}
__device__ __forceinline__ int next_unit_read(SmemTail* tail, bool dynamic, int total, int pair, int num_pairs, UnitCursor& c,
                                              int lane) {
  if (!dynamic) {
    const int u = tile_of(c.rnd, pair, num_pairs);
    ++c.rnd;
    return u < total ? u : -1;
  }
  if (c.first) {
    c.first = false;
    return pair < total ? pair : -1;
  }
  const int slot = c.idx;
  ptx::mbar_wait_acq_cluster(ptx::smem_u32(&tail->rfull[slot]), c.ph);
  const int u = *reinterpret_cast<volatile int32_t*>(&tail->ring[slot]);
  __syncwarp();
  if (lane == 0) ptx::mbar_arrive_cluster(ptx::mapa_u32(ptx::smem_u32(&tail->rempty[slot]), 0));
  if (++c.idx == RING) { c.idx = 0; c.ph ^= 1u; }
  return u;
}

// kMode: 0 = gate|up + SwiGLU (GEMM-1), 1 = down (GEMM-2), 2 = down with the gate-weighted
// scatter fused into the epilogue (vibe_grouped_ffn_scatter; KIND_BF16 only).  kKind: the operand kind (above).
template <int kMode, int kKind>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(num_threads(kMode), 1)
ffn_gemm_kernel(const __grid_constant__ CUtensorMap tmAct, const __grid_constant__ CUtensorMap tmActN,
                const __grid_constant__ CUtensorMap tmW0, const __grid_constant__ CUtensorMap tmW1, const int32_t* __restrict__ offsets, int E_loc,
                int n_total, int k_total, void* __restrict__ out_v, int ld_out,
                const int32_t* __restrict__ row_to_assign, const float* __restrict__ topk_w,
                float* __restrict__ split_part /*NULL: no split-K*/, int* __restrict__ split_cnt,
                unsigned int* __restrict__ unit_ctr /*NULL: static tile assignment*/, const __grid_constant__ FfnAux aux) {
  static_assert(kMode != 2 || kKind == KIND_BF16, "the fused scatter epilogue exists for the bf16 kind only");
  constexpr bool kGateUp = (kMode == 0);
  constexpr bool kMx = (kKind == KIND_MXF8);
  constexpr bool kF8 = (kKind == KIND_F8);
  constexpr int BK = bk_of(kKind);          // K elements per smem stage
  constexpr int UMMA_K = umma_k_of(kKind);
  constexpr int TNk = tn_of(kKind);         // tokens per tile / TMEM columns per accumulator stage
  constexpr int TALIGN = talign_of(kKind);  // block-scaled: token tiles start on an even scale-factor row block
  constexpr int FB = kGateUp ? 128 : 256;   // output features per pair tile
  constexpr int FC = FB / 2;                // ... per CTA
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  float* xchg = reinterpret_cast<float*>(smem + (size_t)STAGES * STAGE_BYTES);
  float* sx_all = reinterpret_cast<float*>(smem + (size_t)STAGES * STAGE_BYTES + XCHG_BYTES);
  SmemTail* tail = reinterpret_cast<SmemTail*>(smem + (size_t)STAGES * STAGE_BYTES + XCHG_BYTES + SX_BYTES);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = ptx::cluster_ctarank();      // 0 = leader (issues the MMAs)
  const int pair = blockIdx.x >> 1, num_pairs = gridDim.x >> 1;
  const int NB = (n_total + FB - 1) / FB;
  const int KB = k_total / BK;

  // ------------------------------------------------------------------ setup
  // (programmatic dependent launch: this grid's set-up below overlaps the tail of the preceding kernel; nothing
  // that kernel wrote -- offsets, Xp or H -- is read before griddep_wait)
  if (warp == 0 && lane == 0) {
    ptx::prefetch_tensormap(&tmAct);
    ptx::prefetch_tensormap(&tmActN);
    ptx::prefetch_tensormap(&tmW0);
    if (kGateUp) ptx::prefetch_tensormap(&tmW1);
    if (kMx) {
      ptx::prefetch_tensormap(&aux.tmSFW);
      ptx::prefetch_tensormap(&aux.tmSFB);
    }
    for (int s = 0; s < STAGES; ++s) {
      ptx::mbar_init(ptx::smem_u32(&tail->full[s]), 1);
      ptx::mbar_init(ptx::smem_u32(&tail->empty[s]), 1);
    }
    for (int a = 0; a < 2; ++a) {
      ptx::mbar_init(ptx::smem_u32(&tail->tfull[a]), 1);
      ptx::mbar_init(ptx::smem_u32(&tail->tempty[a]), 2 * (num_threads(kMode) / 32 - 2));   // epilogue warps of the pair
    }
    for (int r = 0; r < RING; ++r) {
      ptx::mbar_init(ptx::smem_u32(&tail->rfull[r]), 1);
      // readers of a slot: the peer's producer warp, the leader's MMA warp, the epilogue warps of both CTAs
      ptx::mbar_init(ptx::smem_u32(&tail->rempty[r]), 2 + 2 * (num_threads(kMode) / 32 - 2));
    }
    ptx::fence_barrier_init();
  } else if (warp == 1) {
    ptx::tmem_alloc_2sm(ptx::smem_u32(&tail->tmem_base), TMEM_COLS);
    ptx::tmem_relinquish_2sm();
  } else if (warp == 2) {
    // segment starts + exclusive scan of token tiles per slot (warp-shuffle scan, 32 slots a step)
    ptx::griddep_wait();
    int carry = 0;
    for (int base = 0; base < E_loc; base += 32) {
      const int e = base + lane;
      int lo = 0, hi = 0;
      if (e < E_loc) {
        lo = offsets[e];
        hi = offsets[e + 1];
        tail->off[e] = lo;
      }
      // An expert's rows are cut into nt EQUAL token tiles (not 256, 256, ..., remainder): the pairs
      // that share its weight tile (same feature block, other token tiles) and its activation tile
      // (same token tile, other feature blocks) then run K steps of the same length and stay in
      // step, which is what lets L2 serve the second reader.  With a short last tile the readers
      // drift apart by more than L2 holds and DRAM traffic doubles (measured, profiles/).
      const int nt = (hi - lo + TNk - 1) / TNk;
      if (e < E_loc) tail->tsz[e] = nt > 0 ? ((((hi - lo + nt - 1) / nt) + TALIGN - 1) & ~(TALIGN - 1)) : TNk;
      int inc = nt;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int n = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += n;
      }
      if (e < E_loc) tail->cum[e] = carry + inc - nt;
      carry += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) {
      tail->cum[E_loc] = carry;
      tail->off[E_loc] = offsets[E_loc];
      tail->total_t_tiles = carry;
      // Split-K covers the LAST, partly filled round of tiles: with total = q * pairs + r tiles, the r tiles of
      // the last round would occupy r pairs for a whole tile time while the others idle (r = 34 of 74 at 8 x 512
      // rows of the C1 down projection: 14 % of the kernel).  When r <= pairs / 2 each of them is cut into
      // S = pairs / r K slices (q = 0 is the few-active-experts case above).
      int S = 1;
      const int total = carry * NB;
      int from = total;
      const int r = total % num_pairs;
      // (only when the last round is a material share of the kernel: at most 7 rounds -- beyond that the dump /
      // fence / re-read of a split tile costs about what the idle pairs would; measured, same-box A/B)
      if (split_part != nullptr && r > 0 && 2 * r <= num_pairs && total / num_pairs <= 6 && num_pairs <= SPLIT_MAX_UNITS) {
        S = max(1, min(min(num_pairs / r, SPLIT_MAX), KB / SPLIT_MIN_STEPS));
        if (S > 1) from = total - r;
      }
      tail->split_from = from;
      tail->split = S;
    }
  }
  if (warp != 2) ptx::griddep_wait();
  ptx::tc_fence_before();
  __syncthreads();
  ptx::cluster_sync_all();      // the peer's barriers are initialised before anything signals them
  ptx::tc_fence_after();

  const uint32_t tmem_base = tail->tmem_base;
  const int S = tail->split;                               // K slices of a split tile
  const int split_from = tail->split_from;                 // tiles below are whole units, tiles from here on S units each
  const int total_units = split_from + (tail->total_t_tiles * NB - split_from) * S;    // a unit = (tile, K slice)

  if (warp == 0) {
    // ================================================================ TMA producer (both CTAs)
    // The WHOLE warp walks the tile list (warp-uniform control flow and operands); one elected
    // lane issues the expect_tx and the TMA instructions.
    {
      // Both operands are re-read through L2: an activation tile by every feature block of its
      // expert, a weight tile by the pairs working on the other token tiles of the same expert.
      // Those pairs are NOT in lock-step (tile costs differ with the ragged N), so a weight line
      // must survive a few microseconds: evict_first on the weights doubled the DRAM reads
      // (measured, profiles/), evict_last keeps them at the algorithmic bytes.
      const uint64_t pol_act = ptx::policy_evict_last();
      const uint64_t pol_w = ptx::policy_evict_last();
      const uint32_t smem_base = ptx::smem_u32(smem);
      const uint32_t full0 = ptx::mapa_u32(ptx::smem_u32(&tail->full[0]), 0);   // the leader's barriers
      TileCursor cur;
      int stage = 0;
      uint32_t phase = 0;
      UnitCursor uc;
      for (;;) {
        const int unit = rank == 0 ? next_unit_fetch(tail, unit_ctr, total_units, pair, num_pairs, uc, lane)
                                   : next_unit_read(tail, unit_ctr != nullptr, total_units, pair, num_pairs, uc, lane);
        if (unit < 0) break;
        int f_blk, t_blk;
        const bool is_split = unit >= split_from;
        const int tile = is_split ? split_from + (unit - split_from) / S : unit;
        const int slice = is_split ? (unit - split_from) % S : 0, nsl = is_split ? S : 1;
        const int kb_lo = slice * KB / nsl, kb_hi = (slice + 1) * KB / nsl;
        cur.decode(tail, tile, NB, f_blk, t_blk);
        const int e = cur.e;
        const int tsz = tail->tsz[e];
        const int row0 = tail->off[e] + t_blk * tsz;
        const int n_rows = min(tsz, tail->off[e + 1] - row0);
        const int half = ((n_rows + 15) >> 4) << 3;          // UMMA N / 2: this CTA's share of the columns
        const int row_b = row0 + (int)rank * half;
        const int n0 = f_blk * FB + (int)rank * FC;
        // a tile of at most 2 * NARROW_ROWS tokens loads the small activation box (4 KB instead of 16 KB a stage)
        const bool narrow = half <= NARROW_ROWS;
        const CUtensorMap* tm_b = narrow ? &tmActN : &tmAct;
        // Block-scaled kind: the tile's token scales.  A TMA box must start on a 16-byte boundary of global
        // memory (measured: a start at 4 or 8 bytes faults), i.e. on a multiple of 4 row blocks, while a tile starts
        // on any EVEN row block: fetch the aligned {4 row blocks x 32 rows} chunks that cover the tile (at most 2)
        // and point the MMA (rb0 & 3) = 0 or 2 columns into them (measured: the scale-factor TMEM address of the
        // MMA and the destination of tcgen05.cp must be even columns -- an odd one raises "misaligned address").
        const int rb0 = row0 >> 5;
        const int sf_chunks = ((rb0 & 3) + ((half + 15) >> 4) + 3) >> 2;
        const uint32_t tx_bytes = 2u * ((uint32_t)A_BYTES + (uint32_t)(narrow ? NARROW_ROWS * 128 : (kMx ? B_BYTES_MX : B_BYTES)) +
                                        (kMx ? 512u + 512u * (uint32_t)sf_chunks : 0u));
        for (int kb = kb_lo; kb < kb_hi; ++kb) {
          ptx::mbar_wait(ptx::smem_u32(&tail->empty[stage]), phase ^ 1u);
          if (ptx::elect_one()) {
            if (rank == 0) ptx::mbar_arrive_expect_tx(ptx::smem_u32(&tail->full[stage]), tx_bytes);
            const uint32_t full = full0 + (uint32_t)stage * 8u;
            const uint32_t a_s = smem_base + (uint32_t)stage * STAGE_BYTES;
            const uint32_t b_s = a_s + A_BYTES;
            const int k0 = kb * BK;
            // weights: the bf16 tensors are [E_loc, K, N] (N innermost), the packed e4m3 ones [E_loc, N, K] (K innermost)
            const int c0 = (kKind == KIND_BF16) ? n0 : k0, c1 = (kKind == KIND_BF16) ? k0 : n0;
            const int d0 = (kKind == KIND_BF16) ? 64 : 0, d1 = (kKind == KIND_BF16) ? 0 : 64;     // the second 64-feature atom
            if (kGateUp) {
              ptx::tma_load_3d_2sm(a_s, &tmW0, full, c0, c1, e, pol_w);                 // gate -> lanes 0..63
              ptx::tma_load_3d_2sm(a_s + ATOM_BYTES, &tmW1, full, c0, c1, e, pol_w);    // up   -> lanes 64..127
            } else {
              ptx::tma_load_3d_2sm(a_s, &tmW0, full, c0, c1, e, pol_w);
              ptx::tma_load_3d_2sm(a_s + ATOM_BYTES, &tmW0, full, c0 + d0, c1 + d1, e, pol_w);
            }
            ptx::tma_load_2d_2sm(b_s, tm_b, full, k0, row_b, pol_act);
            if (kMx) {
              const int wchunk = (e * KB + kb) * aux.wchunks + n0 / FC;
              ptx::tma_load_2d_2sm(a_s + SFA_OFF, &aux.tmSFW, full, 0, wchunk, pol_w);
              for (int c = 0; c < sf_chunks; ++c)
                ptx::tma_load_3d_2sm(a_s + SFB_OFF + c * 512, &aux.tmSFB, full, (rb0 & ~3) + 4 * c, 0, kb, pol_act);
            }
          }
          __syncwarp();
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
      }
    }
  }
  else if (warp == 1) {
    // ================================================================ UMMA issuer (leader CTA)
    // The whole warp runs the loop; one elected lane issues the MMAs and the commits (always the
    // same lane: tcgen05.commit tracks the MMAs of the issuing thread).
    if (rank == 0) {
      constexpr uint32_t idesc0 = kKind == KIND_BF16 ? ptx::make_idesc_bf16_f32(256, 0, /*a_mn=*/true, /*b_mn=*/false)
                                  : kMx            ? ptx::make_idesc_mxe4m3(256, 0)
                                                   : ptx::make_idesc_e4m3_f32(256, 0);
      // descriptor = constant high word | low word (start address >> 4 in bits [0,14), LBO in [16,30))
      constexpr uint32_t DESC_HI = (1024u >> 4) | (1u << 14) | (2u << 29);
      // A: bf16 weights are MN-major SW128 (LBO = one 8 KB atom; a K step of 16 rows = 2 swizzle atoms of 1024 B),
      //    packed e4m3 weights K-major SW128 (a K step of 32 elements = 32 bytes inside the 128-byte row);
      // B: K-major SW128 for every kind (a K step = 32 bytes inside the row)
      constexpr uint32_t A_LBO = (kKind == KIND_BF16) ? (uint32_t)(ATOM_BYTES >> 4) : (16u >> 4);
      constexpr uint32_t A_KSTEP = (kKind == KIND_BF16) ? (uint32_t)(UMMA_K * 128 / 16) : 2u;
      const uint32_t smem_base = ptx::smem_u32(smem);
      const uint32_t a_lo0 = ((smem_base >> 4) & 0x3fffu) | (A_LBO << 16);
      const uint32_t b_lo0 = (((smem_base + A_BYTES) >> 4) & 0x3fffu) | ((16u >> 4) << 16);
      const uint32_t sfa_t = tmem_base + SF_TMEM_COL, sfb_t = tmem_base + SF_TMEM_COL + 4;
      TileCursor cur;
      int stage = 0;
      uint32_t phase = 0;
      int it = 0;
      UnitCursor uc;
      for (;; ++it) {
        const int unit = next_unit_read(tail, unit_ctr != nullptr, total_units, pair, num_pairs, uc, lane);
        if (unit < 0) break;
        int f_blk, t_blk;
        const bool is_split = unit >= split_from;
        const int tile = is_split ? split_from + (unit - split_from) / S : unit;
        const int slice = is_split ? (unit - split_from) % S : 0, nsl = is_split ? S : 1;
        const int kb_lo = slice * KB / nsl, kb_hi = (slice + 1) * KB / nsl;
        cur.decode(tail, tile, NB, f_blk, t_blk);
        const int e = cur.e;
        const int tsz = tail->tsz[e];
        const int row0 = tail->off[e] + t_blk * tsz;
        const int n_rows = min(tsz, tail->off[e + 1] - row0);
        const uint32_t n_mma = (uint32_t)((n_rows + 15) >> 4) << 4;
        const uint32_t idesc = idesc0 | ((n_mma >> 3) << 17);
        const uint32_t sf_shift = (uint32_t)(row0 >> 5) & 3u;                    // columns into the aligned scale chunks
        const int sf_chunks = (int)((sf_shift + ((n_mma + 31) >> 5) + 3) >> 2);
        const int acc = it & 1;
        const uint32_t acc_phase = (uint32_t)(it >> 1) & 1u;
        ptx::mbar_wait(ptx::smem_u32(&tail->tempty[acc]), acc_phase ^ 1u);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)acc * TNk;
        for (int kb = kb_lo; kb < kb_hi; ++kb) {
          ptx::mbar_wait(ptx::smem_u32(&tail->full[stage]), phase);
          ptx::tc_fence_after();
          if (ptx::elect_one()) {
            if (kMx) {
              // this stage's scale factors: shared memory -> TMEM of both CTAs, ahead of (and ordered with) its MMAs
              const uint32_t sf_s = smem_base + (uint32_t)stage * STAGE_BYTES;
              ptx::tmem_cp_32x128b_warpx4_2sm(sfa_t, ptx::make_smem_desc_rows16(sf_s + SFA_OFF));
              for (int c = 0; c < sf_chunks; ++c)
                ptx::tmem_cp_32x128b_warpx4_2sm(sfb_t + 4u * (uint32_t)c, ptx::make_smem_desc_rows16(sf_s + SFB_OFF + 512u * (uint32_t)c));
            }
            const uint32_t a_lo = a_lo0 + (uint32_t)stage * (STAGE_BYTES >> 4);
            const uint32_t b_lo = b_lo0 + (uint32_t)stage * (STAGE_BYTES >> 4);
#pragma unroll
            for (int k = 0; k < BK / UMMA_K; ++k) {
              const uint64_t da = ((uint64_t)DESC_HI << 32) | (uint64_t)(a_lo + (uint32_t)k * A_KSTEP);
              const uint64_t db = ((uint64_t)DESC_HI << 32) | (uint64_t)(b_lo + (uint32_t)k * 2u);
              const uint32_t accum = (uint32_t)((kb > kb_lo) | (k != 0));
              if (kKind == KIND_BF16)
                ptx::umma_bf16_2sm(d_tmem, da, db, idesc, accum);
              else if (kMx)
                ptx::umma_mxf8_2sm(d_tmem, da, db, idesc | ((uint32_t)k << 29) | ((uint32_t)k << 4), accum, sfa_t, sfb_t + sf_shift);
              else
                ptx::umma_f8_2sm(d_tmem, da, db, idesc, accum);
            }
            ptx::umma_commit_2sm_mc(ptx::smem_u32(&tail->empty[stage]), 3);   // frees the stage in both CTAs
            if (kb == kb_hi - 1)
              ptx::umma_commit_2sm_mc(ptx::smem_u32(&tail->tfull[acc]), 3);   // accumulator ready in both CTAs
          }
          __syncwarp();
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
      }
    }
  }
  else {
    // ================================================================ epilogue (warps 2.., both CTAs)
    const int q = warp & 3;  // TMEM lane quarter this warp may access
    const int blk_par = (warp - 2) >> 2;   // down projection: which 32-column blocks (even / odd) are mine
    TileCursor cur;
    int it = 0;
    UnitCursor uc;
    for (;; ++it) {
      const int unit = next_unit_read(tail, unit_ctr != nullptr, total_units, pair, num_pairs, uc, lane);
      if (unit < 0) break;
      int f_blk, t_blk;
      const bool is_split = unit >= split_from;
      const int tile = is_split ? split_from + (unit - split_from) / S : unit;
      cur.decode(tail, tile, NB, f_blk, t_blk);
      const int e = cur.e;
      const int tsz = tail->tsz[e];
      const int row0 = tail->off[e] + t_blk * tsz;
      const int n_rows = min(tsz, tail->off[e + 1] - row0);
      const int acc = it & 1;
      const uint32_t acc_phase = (uint32_t)(it >> 1) & 1u;
      // fused scatter: destination row and gate weight of this tile's tokens go to this warp's
      // 2 KB slice of the (otherwise unused) exchange buffer while the MMAs of the tile still run
      float* sc_wt = xchg + (warp - 2) * (2 * TN);
      int* sc_asg = reinterpret_cast<int*>(sc_wt + TN);
      if (kMode == 2) {
        __syncwarp();                       // the previous tile's reads of the slice are done
#pragma unroll
        for (int b = 0; b < TN / 32; ++b) {
          const int c = b * 32 + lane;
          const int a = (c < n_rows) ? __ldg(row_to_assign + row0 + c) : -1;
          sc_asg[c] = a;
          sc_wt[c] = (a >= 0) ? __ldg(topk_w + a) : 0.0f;
        }
        __syncwarp();
      }
      // KIND_F8 GEMM-1: the tile's row scales sx go to this warp's slice while the MMAs of the tile still run
      float* sx = sx_all + (warp - 2) * TN;
      if (kF8 && kGateUp) {
        __syncwarp();
#pragma unroll
        for (int b = 0; b < TN / 32; ++b) {
          const int c = b * 32 + lane;
          sx[c] = (c < n_rows) ? __ldg(aux.row_scale + row0 + c) : 0.0f;
        }
        __syncwarp();
      }
      const float se0 = kF8 ? __ldg(aux.sw0 + e) : 1.0f;
      const float se1 = (kF8 && kGateUp) ? __ldg(aux.sw1 + e) : 1.0f;
      const float she = kF8 ? __ldg(aux.h_scale + e) : 1.0f;
      const float inv_sh = kF8 ? 1.0f / she : 1.0f;
      // lanes 0..63 gate (q = 0,1), lanes 64..127 up (q = 2,3) of the same 64 features (GEMM-1); 128 features (GEMM-2)
      const int feat = kGateUp ? f_blk * FB + (int)rank * FC + (q & 1) * 32 + lane : f_blk * FB + (int)rank * FC + q * 32 + lane;
      const bool feat_ok = feat < n_total;

      // ---- what a kind does with finished accumulator values -------------------------------------------------
      // GEMM-1, one element: the accumulators (gate, up) of token column `col` -> the value stored for H
      auto h_of = [&](float g, float u, int col) -> float {
        if (kF8) {
          const float sxi = sx[col];
          return swiglu(g * (sxi * se0), u * (sxi * se1)) * inv_sh;
        }
        return swiglu(g, u);       // KIND_MXF8: the block scales were applied by the tensor core
      };
      // GEMM-1, a finished 32-feature x 32-token block of H (h[i] = token column cbase + i of this lane's feature)
      auto store_h = [&](float (&h)[32], int cbase) {
        if (kMx) {
          // Q7: this warp's 32 lanes are the 32 features of ONE scale block of H.  Per token column: the block's
          // absmax (non-negative floats order like their bit patterns: one redux.sync), e = smallest exponent
          // with amax <= 448 * 2^e (448 = 1.75 * 2^8: e = x - 8, +1 if the mantissa exceeds 1.75), the exact
          // division by 2^e as a multiplication, and lane i keeps the byte of column i.
          uint32_t my_byte = 127u;
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            const uint32_t bits = __reduce_max_sync(0xffffffffu, __float_as_uint(fabsf(h[i])));
            int ex = (int)(bits >> 23) - 127 - 8 + ((bits & 0x7fffffu) > 0x600000u ? 1 : 0);
            ex = bits == 0u ? 0 : max(ex, -127);
            h[i] *= __uint_as_float((uint32_t)(127 - ex) << 23);
            if (lane == i) my_byte = (uint32_t)(ex + 127);
          }
          const int r = row0 + cbase + lane;
          const int fb = feat >> 5;      // warp-uniform
          if (feat_ok && cbase + lane < n_rows)
            aux.hsf[((size_t)((fb >> 2) * 32 + (r & 31)) * (size_t)aux.Rb + (size_t)(r >> 5)) * 4 + (size_t)(fb & 3)] = (uint8_t)my_byte;
        }
        if (kKind == KIND_BF16)
          store_block_T(h, reinterpret_cast<__nv_bfloat16*>(out_v), (size_t)ld_out, row0 + cbase, n_rows - cbase, feat, feat_ok, lane);
        else
          store_block_T_e4m3(h, reinterpret_cast<uint8_t*>(out_v), (size_t)ld_out, row0 + cbase, n_rows - cbase, feat, feat_ok, lane);
      };
      // GEMM-2, a finished 32-feature x 32-token block of Y
      auto store_y = [&](float (&v)[32], int c0) {
        if (kF8) {
#pragma unroll
          for (int i = 0; i < 32; ++i) v[i] *= she * se0;
        }
        if (kMode == 2)
          store_block_T_scatter(v, reinterpret_cast<__nv_bfloat16*>(out_v), (size_t)ld_out, feat, feat_ok, lane, sc_wt + c0, sc_asg + c0);
        else
          store_block_T(v, reinterpret_cast<__nv_bfloat16*>(out_v), (size_t)ld_out, row0 + c0, n_rows - c0, feat, feat_ok, lane);
      };

      ptx::mbar_wait(ptx::smem_u32(&tail->tfull[acc]), acc_phase);
      ptx::tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)acc * TNk;
      if (is_split) {
        // ------------------------------------------------------------ split-K unit
        // (1) dump this warp's part of the fp32 accumulator: part[unit][column][rank * 128 + TMEM lane]
        float* mypart = split_part + ((size_t)(unit - split_from) * TN) * 256 + rank * 128 + q * 32 + lane;
        for (int c0 = kGateUp ? 0 : blk_par * 32; c0 < n_rows; c0 += kGateUp ? 32 : 64) {
          uint32_t a[32];
          ptx::tmem_ld_32x32(taddr + c0, a);
          ptx::tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 32; ++i) __stcg(mypart + (size_t)(c0 + i) * 256, __uint_as_float(a[i]));
        }
        // the accumulator stage is free again
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive_cluster(ptx::mapa_u32(ptx::smem_u32(&tail->tempty[acc]), 0));
        // (2) arrive on the counter of this tile portion; the last of its S (x 2: gate and up warp) arrivals finishes it
        const int role = kGateUp ? (q & 1) : (warp - 2);
        int* cnt = split_cnt + ((tile - split_from) * 2 + (int)rank) * 8 + role;
        const int expect = kGateUp ? 2 * S : S;
        __threadfence();
        int last = 0;
        if (lane == 0) {
          last = (atomicAdd(cnt, 1) == expect - 1);
          if (last) *cnt = 0;               // re-armed for the next call on this workspace
        }
        last = __shfl_sync(0xffffffffu, last, 0);
        if (last) {
          __threadfence();
          // (3) sum the S partials in slice order, then the normal epilogue on the sum
          const float* p0 = split_part + ((size_t)(tile - split_from) * S * TN) * 256 + rank * 128;
          if (kGateUp) {
            const float* pg = p0 + (q & 1) * 32 + lane;        // gate: TMEM lanes 0..63, up: the same feature + 64
            for (int c0 = 0; c0 < n_rows; c0 += 32) {
              // slice loop OUTSIDE, the 32 columns unrolled inside: 64 independent L2 loads in flight per slice
              float g[32], u[32];
#pragma unroll
              for (int i = 0; i < 32; ++i) g[i] = u[i] = 0.0f;
              for (int sl = 0; sl < S; ++sl) {
                const float* pc = pg + ((size_t)sl * TN + (size_t)c0) * 256;
#pragma unroll
                for (int i = 0; i < 32; ++i) {
                  g[i] += __ldcg(pc + (size_t)i * 256);
                  u[i] += __ldcg(pc + (size_t)i * 256 + 64);
                }
              }
#pragma unroll
              for (int i = 0; i < 32; ++i) g[i] = h_of(g[i], u[i], c0 + i);
              store_h(g, c0);
            }
          } else {
            const float* pv = p0 + q * 32 + lane;
            for (int c0 = blk_par * 32; c0 < n_rows; c0 += 64) {
              float v[32];
#pragma unroll
              for (int i = 0; i < 32; ++i) v[i] = 0.0f;
              for (int sl = 0; sl < S; ++sl) {
                const float* pc = pv + ((size_t)sl * TN + (size_t)c0) * 256;
#pragma unroll
                for (int i = 0; i < 32; ++i) v[i] += __ldcg(pc + (size_t)i * 256);
              }
              store_y(v, c0);
            }
          }
        }
        continue;
      }
      if (kGateUp) {
        // Per 64 columns: the gate warp finishes columns 0..31 (needs the partner's up block),
        // the up warp finishes columns 32..63 (needs the partner's gate block).
        const bool is_up = q >= 2;
        float* mine = xchg + ((q & 1) * 2 + (is_up ? 1 : 0)) * 1024;      // block I publish  [col][lane]
        float* theirs = xchg + ((q & 1) * 2 + (is_up ? 0 : 1)) * 1024;    // block my partner publishes
        const uint32_t bar_id = 1 + (q & 1);
        for (int c0 = 0; c0 < n_rows; c0 += 64) {
          uint32_t a[32], b[32];
          ptx::tmem_ld_32x32(taddr + c0, a);
          ptx::tmem_ld_32x32(taddr + c0 + 32, b);
          ptx::tmem_ld_wait();
          // publish the block the partner finishes: gate warp -> its gate of cols 32..63; up warp -> its up of cols 0..31
#pragma unroll
          for (int i = 0; i < 32; ++i) mine[i * 32 + lane] = __uint_as_float(is_up ? a[i] : b[i]);
          ptx::named_bar_sync(bar_id, 64);
          const int cbase = c0 + (is_up ? 32 : 0);
          float h[32];
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            const float o = theirs[i * 32 + lane];
            h[i] = is_up ? h_of(o, __uint_as_float(b[i]), cbase + i) : h_of(__uint_as_float(a[i]), o, cbase + i);
          }
          ptx::named_bar_sync(bar_id, 64);     // both blocks consumed before the next publish
          store_h(h, cbase);
        }
      } else {
#pragma unroll
        for (int b = 0; b < TNk / 32; ++b) {
          const int c0 = b * 32;
          if (c0 >= n_rows) break;
          if ((b & 1) != blk_par) continue;
          uint32_t a[32];
          ptx::tmem_ld_32x32(taddr + c0, a);
          ptx::tmem_ld_wait();
          float v[32];
#pragma unroll
          for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(a[i]);
          store_y(v, c0);
        }
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive_cluster(ptx::mapa_u32(ptx::smem_u32(&tail->tempty[acc]), 0));
    }
  }

  // ------------------------------------------------------------------ teardown
  ptx::tc_fence_before();
  __syncthreads();
  ptx::griddep_launch();        // all tiles of this CTA are done: the next kernel's CTAs may become resident
  ptx::cluster_sync_all();      // neither CTA frees TMEM / exits while the peer still uses the pair
  if (warp == 1) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc_2sm(tmem_base, TMEM_COLS);
  }
}

// ---------------------------------------------------------------------------------------
// TMA tensor maps (host).  cuTensorMapEncodeTiled is a driver entry point fetched through
// the runtime, so libvibe.so does not link libcuda.  Maps are cached for the process
// lifetime, keyed by (pointer, shape, element type): weights and workspaces are long-lived in serving.
// ---------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  });
  return fn;
}

// element types of the maps: bf16 and one-byte operands with the 128-byte swizzle; 32-bit words without
// swizzle (the scale-factor arrays of the block-scaled kind)
enum MapElem { ELEM_BF16 = 0, ELEM_U8 = 1, ELEM_WORDS = 2 };

struct MapKey {
  const void* ptr;
  uint64_t d0, d1, d2;
  uint32_t b0, b1;
  int elem;
  bool operator==(const MapKey& o) const {
    return ptr == o.ptr && d0 == o.d0 && d1 == o.d1 && d2 == o.d2 && b0 == o.b0 && b1 == o.b1 && elem == o.elem;
  }
};
struct MapKeyHash {
  size_t operator()(const MapKey& k) const {
    size_t h = reinterpret_cast<size_t>(k.ptr);
    h = h * 1315423911u ^ k.d0;
    h = h * 1315423911u ^ k.d1;
    h = h * 1315423911u ^ k.d2;
    h = h * 1315423911u ^ ((uint64_t)k.b0 << 32 | k.b1);
    h = h * 1315423911u ^ (size_t)k.elem;
    return h;
  }
};
std::mutex g_map_mu;
std::unordered_map<MapKey, CUtensorMap, MapKeyHash> g_maps;

// rank 2: dims (d0 inner, d1); rank 3: dims (d0 inner, d1, d2)
vibe_status get_tensor_map(MapElem elem, const void* ptr, uint64_t d0, uint64_t d1, uint64_t d2, uint32_t box0, uint32_t box1,
                           CUtensorMap* out) {
  MapKey key{ptr, d0, d1, d2, box0, box1, (int)elem};
  {
    std::lock_guard<std::mutex> lk(g_map_mu);
    auto it = g_maps.find(key);
    if (it != g_maps.end()) {
      *out = it->second;
      return VIBE_OK;
    }
  }
  EncodeTiledFn enc = get_encode_fn();
  VIBE_REQUIRE(enc != nullptr, VIBE_ERR_CUDA, "cuTensorMapEncodeTiled entry point unavailable (no CUDA driver?)");
  const bool r3 = d2 > 0;
  const uint64_t esz = elem == ELEM_BF16 ? 2 : elem == ELEM_U8 ? 1 : 4;
  cuuint64_t dims[3] = {d0, d1, r3 ? d2 : 1};
  cuuint64_t strides[2] = {d0 * esz, d0 * d1 * esz};
  cuuint32_t box[3] = {box0, box1, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUtensorMap m;
  const CUtensorMapDataType dt = elem == ELEM_BF16 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16
                                 : elem == ELEM_U8 ? CU_TENSOR_MAP_DATA_TYPE_UINT8
                                                   : CU_TENSOR_MAP_DATA_TYPE_UINT32;
  CUresult r = enc(&m, dt, r3 ? 3 : 2, const_cast<void*>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   elem == ELEM_WORDS ? CU_TENSOR_MAP_SWIZZLE_NONE : CU_TENSOR_MAP_SWIZZLE_128B,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  VIBE_REQUIRE(r == CUDA_SUCCESS, VIBE_ERR_CUDA,
               "cuTensorMapEncodeTiled failed (CUresult %d) ptr=%p dims=(%llu,%llu,%llu) box=(%u,%u)", (int)r, ptr,
               (unsigned long long)d0, (unsigned long long)d1, (unsigned long long)d2, box0, box1);
  {
    std::lock_guard<std::mutex> lk(g_map_mu);
    if (g_maps.size() > 4096) g_maps.clear();
    g_maps[key] = m;
  }
  *out = m;
  return VIBE_OK;
}

// the opt-in to > 48 KB of dynamic shared memory is per device: once for each device this process uses
vibe_status set_smem_attrs() {
  static std::mutex mu;
  static bool done[kMaxDevices] = {};
  const int dev = current_device();
  std::lock_guard<std::mutex> lk(mu);
  if (done[dev]) return VIBE_OK;
  const int b = (int)SMEM_BYTES;
  VIBE_CUDA(cudaFuncSetAttribute(ffn_gemm_kernel<0, KIND_BF16>, cudaFuncAttributeMaxDynamicSharedMemorySize, b));
  VIBE_CUDA(cudaFuncSetAttribute(ffn_gemm_kernel<1, KIND_BF16>, cudaFuncAttributeMaxDynamicSharedMemorySize, b));
  VIBE_CUDA(cudaFuncSetAttribute(ffn_gemm_kernel<2, KIND_BF16>, cudaFuncAttributeMaxDynamicSharedMemorySize, b));
  VIBE_CUDA(cudaFuncSetAttribute(ffn_gemm_kernel<0, KIND_F8>, cudaFuncAttributeMaxDynamicSharedMemorySize, b));
  VIBE_CUDA(cudaFuncSetAttribute(ffn_gemm_kernel<1, KIND_F8>, cudaFuncAttributeMaxDynamicSharedMemorySize, b));
  VIBE_CUDA(cudaFuncSetAttribute(ffn_gemm_kernel<0, KIND_MXF8>, cudaFuncAttributeMaxDynamicSharedMemorySize, b));
  VIBE_CUDA(cudaFuncSetAttribute(ffn_gemm_kernel<1, KIND_MXF8>, cudaFuncAttributeMaxDynamicSharedMemorySize, b));
  done[dev] = true;
  return VIBE_OK;
}

// split-K workspace of a call: partial buffer + the counters of the two launches (NULL pointers: split-K off)
struct SplitWs {
  float* part = nullptr;
  int* cnt1 = nullptr;
  int* cnt2 = nullptr;
  unsigned int* ctr1 = nullptr;   // next-unit counters of the dynamic tile scheduler
  unsigned int* ctr2 = nullptr;
};
vibe_status split_ws(void* ws, size_t ws_bytes, bool ws_zeroed, cudaStream_t st, SplitWs* out) {
  if (ws != nullptr && ws_bytes >= SPLIT_WS_BYTES && (reinterpret_cast<uintptr_t>(ws) & 15u) == 0) {
    out->part = reinterpret_cast<float*>(ws);
    out->cnt1 = reinterpret_cast<int*>(reinterpret_cast<char*>(ws) + SPLIT_PART_BYTES);
    out->cnt2 = out->cnt1 + SPLIT_COUNTERS;
    out->ctr1 = reinterpret_cast<unsigned int*>(out->cnt2 + SPLIT_COUNTERS);
    out->ctr2 = out->ctr1 + 8;

    if (!ws_zeroed) VIBE_CUDA(cudaMemsetAsync(out->cnt1, 0, SPLIT_CNT_BYTES, st));
  }
  return VIBE_OK;
}

// the two launches of one FFN: gate|up + SwiGLU, then down (kDownMode = 1, or 2 with the fused scatter)
template <int kKind, int kDownMode>
vibe_status launch_pair(const CUtensorMap& tmX, const CUtensorMap& tmXN, const CUtensorMap& tmW1, const CUtensorMap& tmW3,
                        const CUtensorMap& tmH, const CUtensorMap& tmHN, const CUtensorMap& tmW2, const int32_t* offsets,
                        int E_loc, int d, int f, void* H, void* Y, const int32_t* row_to_assign, const float* topk_w,
                        const SplitWs& sw, const FfnAux& aux1, const FfnAux& aux2, cudaStream_t st) {
  vibe_status sa = set_smem_attrs();
  if (sa != VIBE_OK) return sa;
  const int grid = num_sms() & ~1;   // CTA pairs (clusters of 2)
  // both launches carry the programmatic-dependent-launch attribute (see the kernel's set-up)
  const int32_t* no_map = nullptr;
  const float* no_w = nullptr;
  // dynamic hand-out of tiles only where a tile is long enough to hide the fetch (one atomic round trip plus two
  // cluster-scope barrier hops per tile, ~1.5 us): at least DYN_MIN_STEPS K stages per tile.  Short-K launches (the
  // C2 shape: 32 / 12 stages) keep the static assignment -- measured 4 % faster there, while the long-K launches of C1
  // gain 1-2 % in time and drop from 1.52 x to 1.09 x the algorithmic DRAM bytes.
  constexpr int DYN_MIN_STEPS = 48;
  unsigned int* ctr1 = (d / bk_of(kKind) >= DYN_MIN_STEPS) ? sw.ctr1 : nullptr;
  unsigned int* ctr2 = (f / bk_of(kKind) >= DYN_MIN_STEPS) ? sw.ctr2 : nullptr;
  cudaError_t le = launch_pdl(ffn_gemm_kernel<0, kKind>, dim3(grid), dim3(num_threads(0)), SMEM_BYTES, st, tmX, tmXN, tmW1, tmW3,
                              offsets, E_loc, f, d, H, f, no_map, no_w, sw.part, sw.cnt1, ctr1, aux1);
  VIBE_REQUIRE(le == cudaSuccess, VIBE_ERR_CUDA, "ffn_gemm_kernel<gate_up> launch failed: %s", cudaGetErrorString(le));
  VIBE_LAUNCH_CHECK("ffn_gemm_kernel<gate_up>");
  le = launch_pdl(ffn_gemm_kernel<kDownMode, kKind>, dim3(grid), dim3(num_threads(kDownMode)), SMEM_BYTES, st, tmH, tmHN, tmW2,
                  tmW2, offsets, E_loc, d, f, Y, d, row_to_assign, topk_w, sw.part, sw.cnt2, ctr2, aux2);
  VIBE_REQUIRE(le == cudaSuccess, VIBE_ERR_CUDA, "ffn_gemm_kernel<down> launch failed: %s", cudaGetErrorString(le));
  VIBE_LAUNCH_CHECK("ffn_gemm_kernel<down>");
  return VIBE_OK;
}

}  // namespace

size_t grouped_ffn_ws_bytes() { return SPLIT_WS_BYTES; }
vibe_status grouped_ffn_zero_counters(void* ws, cudaStream_t st) {
  VIBE_CUDA(cudaMemsetAsync(reinterpret_cast<char*>(ws) + SPLIT_PART_BYTES, 0, SPLIT_CNT_BYTES, st));
  return VIBE_OK;
}

// ws (may be NULL or short: split-K is then off): SPLIT_WS_BYTES bytes; ws_zeroed: the caller has already zeroed the
// counters behind the partial buffer on this stream (the layer entries do it before the route kernel so that no
// memset sits between the permutation and the FFN kernels, which are chained by programmatic dependent launch)
vibe_status grouped_ffn_impl(const void* Xp, const int32_t* offsets, int E_loc, int R_cap, int d, int f,
                             const void* W1, const void* W3, const void* W2, void* H_ws, void* Y,
                             cudaStream_t st, const int32_t* row_to_assign, const float* topk_w, void* ws,
                             size_t ws_bytes, bool ws_zeroed) {
  constexpr int BK = bk_of(KIND_BF16);
  CUtensorMap tmX, tmH, tmXN, tmHN, tmW1, tmW3, tmW2;
  vibe_status s;
  // activations [R_cap, K] K innermost: boxes of 64 K x (128 | 32) rows; weights [E_loc, K, N] N innermost: 64 N x 64 K
  if ((s = get_tensor_map(ELEM_BF16, Xp, d, R_cap, 0, BK, TN / 2, &tmX)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_BF16, H_ws, f, R_cap, 0, BK, TN / 2, &tmH)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_BF16, Xp, d, R_cap, 0, BK, NARROW_ROWS, &tmXN)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_BF16, H_ws, f, R_cap, 0, BK, NARROW_ROWS, &tmHN)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_BF16, W1, f, d, E_loc, 64, BK, &tmW1)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_BF16, W3, f, d, E_loc, 64, BK, &tmW3)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_BF16, W2, d, f, E_loc, 64, BK, &tmW2)) != VIBE_OK) return s;
  SplitWs sw;
  if ((s = split_ws(ws, ws_bytes, ws_zeroed, st, &sw)) != VIBE_OK) return s;
  const FfnAux none{};
  if (row_to_assign != nullptr)
    return launch_pair<KIND_BF16, 2>(tmX, tmXN, tmW1, tmW3, tmH, tmHN, tmW2, offsets, E_loc, d, f, H_ws, Y, row_to_assign, topk_w,
                                     sw, none, none, st);
  return launch_pair<KIND_BF16, 1>(tmX, tmXN, tmW1, tmW3, tmH, tmHN, tmW2, offsets, E_loc, d, f, H_ws, Y, nullptr, nullptr, sw,
                                   none, none, st);
}

// KIND_F8 (readings Q1-Q4): packed weights [E_loc, N, K] (K innermost), per-row / per-expert / static H scales
vibe_status grouped_ffn_fp8_impl(const void* Xq, const float* row_scale, const int32_t* offsets, int E_loc, int R_cap,
                                 int d, int f, const void* W1q, const float* s1, const void* W3q, const float* s3,
                                 const void* W2q, const float* s2, const float* h_scale, void* Hq, void* Y,
                                 cudaStream_t st, void* ws, size_t ws_bytes, bool ws_zeroed) {
  constexpr int BK = bk_of(KIND_F8);
  CUtensorMap tmX, tmH, tmXN, tmHN, tmW1, tmW3, tmW2;
  vibe_status s;
  if ((s = get_tensor_map(ELEM_U8, Xq, d, R_cap, 0, BK, TN / 2, &tmX)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_U8, Hq, f, R_cap, 0, BK, TN / 2, &tmH)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_U8, Xq, d, R_cap, 0, BK, NARROW_ROWS, &tmXN)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_U8, Hq, f, R_cap, 0, BK, NARROW_ROWS, &tmHN)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_U8, W1q, d, f, E_loc, BK, 64, &tmW1)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_U8, W3q, d, f, E_loc, BK, 64, &tmW3)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_U8, W2q, f, d, E_loc, BK, 64, &tmW2)) != VIBE_OK) return s;
  SplitWs sw;
  if ((s = split_ws(ws, ws_bytes, ws_zeroed, st, &sw)) != VIBE_OK) return s;
  FfnAux a1{}, a2{};
  a1.row_scale = row_scale;
  a1.sw0 = s1;
  a1.sw1 = s3;
  a1.h_scale = a2.h_scale = h_scale;
  a2.sw0 = s2;
  return launch_pair<KIND_F8, 1>(tmX, tmXN, tmW1, tmW3, tmH, tmHN, tmW2, offsets, E_loc, d, f, Hq, Y, nullptr, nullptr, sw, a1, a2, st);
}

// KIND_MXF8 (readings Q5-Q8).  sf13: joint gate|up weight scales (one 512-byte chunk per expert, K stage and 64
// features: TMEM rows 0..63 = W1's, 64..127 = W3's); sf2: down-projection weight scales (chunk per 128 features);
// xsf / hsf: token scales [K/128][32][Rb] words (hsf is written by GEMM-1 and read by GEMM-2).
vibe_status grouped_ffn_mxfp8_impl(const void* Xq, const void* xsf, const int32_t* offsets, int E_loc, int R_cap, int d,
                                   int f, const void* W1q, const void* W3q, const void* sf13, const void* W2q,
                                   const void* sf2, void* Hq, void* hsf, void* Y, cudaStream_t st, void* ws,
                                   size_t ws_bytes, bool ws_zeroed) {
  constexpr int BK = bk_of(KIND_MXF8);
  constexpr int TNM = tn_of(KIND_MXF8);
  CUtensorMap tmX, tmH, tmXN, tmHN, tmW1, tmW3, tmW2;
  FfnAux a1{}, a2{};
  vibe_status s;
  const int Rb = mx_row_blocks(R_cap);
  if ((s = get_tensor_map(ELEM_U8, Xq, d, R_cap, 0, BK, TNM / 2, &tmX)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_U8, Hq, f, R_cap, 0, BK, TNM / 2, &tmH)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_U8, Xq, d, R_cap, 0, BK, NARROW_ROWS, &tmXN)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_U8, Hq, f, R_cap, 0, BK, NARROW_ROWS, &tmHN)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_U8, W1q, d, f, E_loc, BK, 64, &tmW1)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_U8, W3q, d, f, E_loc, BK, 64, &tmW3)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_U8, W2q, f, d, E_loc, BK, 64, &tmW2)) != VIBE_OK) return s;
  a1.wchunks = f / 64;
  a2.wchunks = d / 128;
  if ((s = get_tensor_map(ELEM_WORDS, sf13, 128, (uint64_t)E_loc * (d / BK) * a1.wchunks, 0, 128, 1, &a1.tmSFW)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_WORDS, sf2, 128, (uint64_t)E_loc * (f / BK) * a2.wchunks, 0, 128, 1, &a2.tmSFW)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_WORDS, xsf, Rb, 32, d / BK, 4, 32, &a1.tmSFB)) != VIBE_OK) return s;
  if ((s = get_tensor_map(ELEM_WORDS, hsf, Rb, 32, f / BK, 4, 32, &a2.tmSFB)) != VIBE_OK) return s;
  a1.hsf = reinterpret_cast<uint8_t*>(hsf);
  a1.Rb = a2.Rb = Rb;
  SplitWs sw;
  if ((s = split_ws(ws, ws_bytes, ws_zeroed, st, &sw)) != VIBE_OK) return s;
  return launch_pair<KIND_MXF8, 1>(tmX, tmXN, tmW1, tmW3, tmH, tmHN, tmW2, offsets, E_loc, d, f, Hq, Y, nullptr, nullptr, sw, a1, a2, st);
}

// the shape / alignment limits of the FFN kernels, checkable before anything is enqueued (the layer entry points
// call this first: "argument errors are detected before any launch")
vibe_status grouped_ffn_limits(const char* who, int E_loc, int d, int f, const void* W1, const void* W3, const void* W2) {
  VIBE_REQUIRE(W1 && W3 && W2, VIBE_ERR_INVALID_ARG, "%s: NULL weight tensor", who);
  VIBE_REQUIRE(d % 64 == 0 && f % 64 == 0, VIBE_ERR_UNSUPPORTED, "%s: d and f must be multiples of 64 (d=%d f=%d)", who, d, f);
  VIBE_REQUIRE(E_loc <= MAX_SLOTS, VIBE_ERR_UNSUPPORTED, "%s: E_loc > %d not implemented", who, MAX_SLOTS);
  VIBE_REQUIRE(aligned16(W1) && aligned16(W3) && aligned16(W2), VIBE_ERR_INVALID_ARG, "%s: weight tensors must be 16-byte aligned", who);
  return VIBE_OK;
}

vibe_status grouped_ffn_check(const void* Xp, const int32_t* offsets, int E_loc, int R_cap, int d, int f,
                              const void* W1, const void* W3, const void* W2, void* H_ws, void* Y) {
  VIBE_REQUIRE(E_loc >= 1 && R_cap >= 1 && d >= 1 && f >= 1, VIBE_ERR_INVALID_ARG,
               "vibe_grouped_ffn: bad sizes E_loc=%d R_cap=%d d=%d f=%d", E_loc, R_cap, d, f);
  VIBE_REQUIRE(Xp && offsets && W1 && W3 && W2 && H_ws && Y, VIBE_ERR_INVALID_ARG, "vibe_grouped_ffn: NULL tensor");
  VIBE_REQUIRE(d % 64 == 0 && f % 64 == 0, VIBE_ERR_UNSUPPORTED,
               "vibe_grouped_ffn: d and f must be multiples of 64 (d=%d f=%d)", d, f);
  VIBE_REQUIRE(E_loc <= MAX_SLOTS, VIBE_ERR_UNSUPPORTED, "vibe_grouped_ffn: E_loc > %d not implemented", MAX_SLOTS);
  VIBE_REQUIRE(aligned16(Xp) && aligned16(W1) && aligned16(W3) && aligned16(W2) && aligned16(H_ws) && aligned16(Y),
               VIBE_ERR_INVALID_ARG, "vibe_grouped_ffn: all tensors must be 16-byte aligned");
  return VIBE_OK;
}

}  // namespace vibe

extern "C" vibe_status vibe_grouped_ffn(const void* Xp, const int32_t* offsets, int32_t E_loc, int32_t R_cap,
                                        int32_t d, int32_t f, const void* W1, const void* W3, const void* W2,
                                        void* H_ws, void* Y, void* ws, size_t ws_bytes, void* stream) {
  using namespace vibe;
  clear_error();
  vibe_status s = grouped_ffn_check(Xp, offsets, E_loc, R_cap, d, f, W1, W3, W2, H_ws, Y);
  if (s != VIBE_OK) return s;
  return grouped_ffn_impl(Xp, offsets, E_loc, R_cap, d, f, W1, W3, W2, H_ws, Y,
                          reinterpret_cast<cudaStream_t>(stream), nullptr, nullptr, ws, ws_bytes, false);
}

extern "C" vibe_status vibe_grouped_ffn_scatter(const void* Xp, const int32_t* offsets, int32_t E_loc, int32_t R_cap,
                                                int32_t d, int32_t f, const void* W1, const void* W3,
                                                const void* W2, const int32_t* row_to_assign, const float* topk_w,
                                                void* H_ws, void* Yw, void* ws, size_t ws_bytes, void* stream) {
  using namespace vibe;
  clear_error();
  vibe_status s = grouped_ffn_check(Xp, offsets, E_loc, R_cap, d, f, W1, W3, W2, H_ws, Yw);
  if (s != VIBE_OK) return s;
  VIBE_REQUIRE(row_to_assign && topk_w, VIBE_ERR_INVALID_ARG, "vibe_grouped_ffn_scatter: NULL row_to_assign / topk_w");
  return grouped_ffn_impl(Xp, offsets, E_loc, R_cap, d, f, W1, W3, W2, H_ws, Yw,
                          reinterpret_cast<cudaStream_t>(stream), row_to_assign, topk_w, ws, ws_bytes, false);
}

extern "C" vibe_status vibe_grouped_ffn_fp8(const void* Xq, const float* row_scale, const int32_t* offsets,
                                            int32_t E_loc, int32_t R_cap, int32_t d, int32_t f, const void* W1q,
                                            const float* s1, const void* W3q, const float* s3, const void* W2q,
                                            const float* s2, const float* h_scale, void* Hq_ws, void* Y,
                                            void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(E_loc >= 1 && R_cap >= 1 && d >= 1 && f >= 1, VIBE_ERR_INVALID_ARG,
               "vibe_grouped_ffn_fp8: bad sizes E_loc=%d R_cap=%d d=%d f=%d", E_loc, R_cap, d, f);
  VIBE_REQUIRE(Xq && row_scale && offsets && W1q && s1 && W3q && s3 && W2q && s2 && h_scale && Hq_ws && Y,
               VIBE_ERR_INVALID_ARG, "vibe_grouped_ffn_fp8: NULL argument");
  VIBE_REQUIRE(d % 128 == 0 && f % 128 == 0, VIBE_ERR_UNSUPPORTED,
               "vibe_grouped_ffn_fp8: d and f must be multiples of 128 (d=%d f=%d)", d, f);
  VIBE_REQUIRE(E_loc <= MAX_SLOTS, VIBE_ERR_UNSUPPORTED, "vibe_grouped_ffn_fp8: E_loc > %d not implemented", MAX_SLOTS);
  VIBE_REQUIRE(aligned16(Xq) && aligned16(W1q) && aligned16(W3q) && aligned16(W2q) && aligned16(Hq_ws) && aligned16(Y),
               VIBE_ERR_INVALID_ARG, "vibe_grouped_ffn_fp8: all tensors must be 16-byte aligned");
  return grouped_ffn_fp8_impl(Xq, row_scale, offsets, E_loc, R_cap, d, f, W1q, s1, W3q, s3, W2q, s2, h_scale, Hq_ws, Y,
                              reinterpret_cast<cudaStream_t>(stream), nullptr, 0, false);
}

extern "C" vibe_status vibe_grouped_ffn_mxfp8(const void* Xq, const void* Xsf, const int32_t* offsets, int32_t E_loc,
                                              int32_t R_cap, int32_t d, int32_t f, const void* W1q, const void* W3q,
                                              const void* sf13, const void* W2q, const void* sf2, void* Hq_ws,
                                              void* Hsf_ws, void* Y, void* stream) {
  using namespace vibe;
  clear_error();
  VIBE_REQUIRE(E_loc >= 1 && R_cap >= 1 && d >= 1 && f >= 1, VIBE_ERR_INVALID_ARG,
               "vibe_grouped_ffn_mxfp8: bad sizes E_loc=%d R_cap=%d d=%d f=%d", E_loc, R_cap, d, f);
  VIBE_REQUIRE(Xq && Xsf && offsets && W1q && W3q && sf13 && W2q && sf2 && Hq_ws && Hsf_ws && Y, VIBE_ERR_INVALID_ARG,
               "vibe_grouped_ffn_mxfp8: NULL argument");
  VIBE_REQUIRE(d % 128 == 0 && f % 128 == 0, VIBE_ERR_UNSUPPORTED,
               "vibe_grouped_ffn_mxfp8: d and f must be multiples of 128 (d=%d f=%d)", d, f);
  VIBE_REQUIRE(E_loc <= MAX_SLOTS, VIBE_ERR_UNSUPPORTED, "vibe_grouped_ffn_mxfp8: E_loc > %d not implemented", MAX_SLOTS);
  VIBE_REQUIRE(aligned16(Xq) && aligned16(Xsf) && aligned16(W1q) && aligned16(W3q) && aligned16(sf13) && aligned16(W2q) &&
                   aligned16(sf2) && aligned16(Hq_ws) && aligned16(Hsf_ws) && aligned16(Y),
               VIBE_ERR_INVALID_ARG, "vibe_grouped_ffn_mxfp8: all tensors must be 16-byte aligned");
  return grouped_ffn_mxfp8_impl(Xq, Xsf, offsets, E_loc, R_cap, d, f, W1q, W3q, sf13, W2q, sf2, Hq_ws, Hsf_ws, Y,
                                reinterpret_cast<cudaStream_t>(stream), nullptr, 0, false);
}
