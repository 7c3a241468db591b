// ffn_fp8.cu -- S8(f) f2: the grouped SwiGLU expert FFN with FP8 (e4m3) operands
// (vibe_grouped_ffn_fp8).  "Precision: FP8" for both evaluated models (Table 2a);
// recipe = DESIGN.md readings Q1-Q4.
//
// Same machine as ffn.cu (swap-AB, 74 CTA pairs, cta_group::2 MMAs of M = 256, warp-uniform TMA /
// MMA loops, equal token tiles, rotated tile assignment, 2 TMEM accumulator stages) with
//   * tcgen05.mma kind::f8f6f4: K = 32 per instruction, 128 one-byte elements per 128-byte smem row,
//     so a K step is 128 deep and moves the same 32 KB per CTA as the bf16 kernel's 64-deep step
//   * weights pre-quantised AND pre-transposed to [E_loc, N, K] (K contiguous) by vibe_fp8_pack_weights:
//     both operands K-major, plain SW128 descriptors
//   * scales on the accumulators in the epilogue: GEMM-1  g = sx[row] s1[e] acc_g, u = sx[row] s3[e] acc_u,
//     h = silu(g) u, Hq = e4m3(h / sh[e]);  GEMM-2  y = sh[e] s2[e] acc -> bf16
//
// kMx = true: the BLOCK-SCALED variant (vibe_grouped_ffn_mxfp8; readings Q5-Q8): tcgen05.mma
// kind::mxf8f6f4.block_scale with one UE8M0 scale per operand row and 32 K elements.  The scales of a K = 128
// stage travel with the stage (weights: one 512-byte chunk already in TMEM order; tokens: a {4 row-blocks x 32
// rows} boxes of the [K/128][32][Rb] word array, which land in TMEM order; a tile that starts on a 64-row boundary
// reads them from column 0 or 2 of its chunk), are copied
// to TMEM by tcgen05.cp ahead of the stage's four MMAs (same issuing thread: ordered with them), and the
// instruction descriptor's scale-factor ids pick the K-block's byte.  Token tiles are multiples of 64 rows and at
// most 192 (2 x 192 accumulator columns + 12 scale columns fit the 512 TMEM columns); no scale arithmetic is left
// in the epilogues; GEMM-1 block-quantises H per row and 32 features (one warp = one block: redux.sync max).
#include <mutex>
#include <unordered_map>
#include <string>
#include <cstring>

#include "common.cuh"
#include "ptx.cuh"

namespace vibe {
namespace {

constexpr int BK = 128;                 // K per smem stage (one 128-byte swizzle atom of e4m3)
constexpr int TN = 256;                 // tokens per tile = max UMMA N
constexpr int UMMA_K = 32;
constexpr int STAGES = 6;
constexpr int ATOM_BYTES = 64 * BK;             // 8 KB : 64 features x 128 K (K-major, SW128)
constexpr int A_BYTES = 2 * ATOM_BYTES;         // 16 KB: this CTA's 128 accumulator lanes
constexpr int B_BYTES = (TN / 2) * BK;          // 16 KB: this CTA's half of the token tile
constexpr int STAGE_BYTES = A_BYTES + B_BYTES;  // 32 KB
constexpr int NARROW_ROWS = 32;                 // rows of the small activation box (per CTA)
constexpr int XCHG_BYTES = 16384;               // gate/up swap: 2 warp pairs x 2 directions x 4 KB
constexpr int SX_BYTES = 4 * TN * 4;            // GEMM-1: the tile's row scales, one 1 KB slice per epilogue warp
// warps: 0 = TMA producer, 1 = MMA issuer, 2.. = epilogue.  GEMM-1 has 4 epilogue warps (its SwiGLU
// epilogue needs ~200 registers per thread); the down projection has 8 -- two per TMEM lane quarter,
// alternating 32-column blocks -- because with a short K loop (f = 768: 12 K steps per tile) one warp
// per quarter could not drain a 256-column accumulator as fast as the tensor pipe fills the next
// (ncu at the C2 shape: tensor pipe 33 % active with 4 warps).
__host__ __device__ constexpr int num_threads(int mode) { return mode == 0 ? 192 : 320; }
constexpr int MAX_SLOTS = 512;
constexpr int TMEM_COLS = 512;
// block-scaled variant: token tile, per-CTA activation bytes of a stage, where the stage keeps its scale factors
constexpr int TN_MX = 192;
constexpr int B_BYTES_MX = (TN_MX / 2) * BK;    // 12 KB
constexpr int SFA_OFF = A_BYTES + B_BYTES_MX;   // 512 B : this CTA's 128 weight rows x 4 K-blocks
constexpr int SFB_OFF = SFA_OFF + 512;          // 1 KB  : up to two 128-row chunks of token scales x 4 K-blocks
static_assert(SFB_OFF + 1024 <= STAGE_BYTES, "scale factors must fit behind the narrower activation tile");
constexpr uint32_t SF_TMEM_COL = 2 * TN_MX;     // columns 384.. : SFA (4) then SFB (8)

struct MxArgs {
  CUtensorMap tmSFB;   // token scales : u32 [K/128][32][Rb]
  CUtensorMap tmSFW;   // weight scales: u32 [chunks][128 words], one 512-byte chunk per (expert, K stage, CTA feature tile)
  uint8_t* hsf;        // GEMM-1: scales of H, written in the token-scale layout (K = f)
  int Rb;              // words per (K stage, lane) row of the token-scale arrays
  int wchunks;         // weight chunks per (expert, K stage)
};

struct SmemTail {
  uint64_t full[STAGES];          // leader CTA: both CTAs' TMA bytes of a stage have landed
  uint64_t empty[STAGES];         // each CTA: the MMAs reading the stage have retired
  uint64_t tfull[2];              // each CTA: accumulator stage complete
  uint64_t tempty[2];             // leader CTA: all 8 epilogue warps of the pair drained it
  uint32_t tmem_base;
  int32_t total_t_tiles;
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

// kMode: 0 = gate|up + SwiGLU (GEMM-1, writes Hq e4m3), 1 = down (GEMM-2, writes Y bf16).
template <int kMode, bool kMx>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(num_threads(kMode), 1)
ffn8_gemm_kernel(const __grid_constant__ CUtensorMap tmAct, const __grid_constant__ CUtensorMap tmActN,
                 const __grid_constant__ CUtensorMap tmW0, const __grid_constant__ CUtensorMap tmW1, const int32_t* __restrict__ offsets, int E_loc,
                 int n_total, int k_total, void* __restrict__ out_v, int ld_out,
                 const float* __restrict__ row_scale /*GEMM-1: sx [R_cap]*/, const float* __restrict__ sw0 /*[E_loc]*/,
                 const float* __restrict__ sw1 /*[E_loc] (GEMM-1: W3)*/, const float* __restrict__ h_scale /*[E_loc]*/,
                 const __grid_constant__ MxArgs mx) {
  constexpr bool kGateUp = (kMode == 0);
  constexpr int TNk = kMx ? TN_MX : TN;      // tokens per tile / TMEM columns per accumulator stage
  constexpr int TALIGN = kMx ? 64 : 16;      // block-scaled: token tiles start on an even scale-factor row block
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
  if (warp == 0 && lane == 0) {
    ptx::prefetch_tensormap(&tmAct);
    ptx::prefetch_tensormap(&tmActN);
    ptx::prefetch_tensormap(&tmW0);
    if (kGateUp) ptx::prefetch_tensormap(&tmW1);
    if (kMx) {
      ptx::prefetch_tensormap(&mx.tmSFW);
      ptx::prefetch_tensormap(&mx.tmSFB);
    }
    for (int s = 0; s < STAGES; ++s) {
      ptx::mbar_init(ptx::smem_u32(&tail->full[s]), 1);
      ptx::mbar_init(ptx::smem_u32(&tail->empty[s]), 1);
    }
    for (int a = 0; a < 2; ++a) {
      ptx::mbar_init(ptx::smem_u32(&tail->tfull[a]), 1);
      ptx::mbar_init(ptx::smem_u32(&tail->tempty[a]), 2 * (num_threads(kMode) / 32 - 2));   // epilogue warps of the pair
    }
    ptx::fence_barrier_init();
  } else if (warp == 1) {
    ptx::tmem_alloc_2sm(ptx::smem_u32(&tail->tmem_base), TMEM_COLS);
    ptx::tmem_relinquish_2sm();
  } else if (warp == 2) {
    // segment starts + exclusive scan of token tiles per slot (warp-shuffle scan, 32 slots a step)
    ptx::griddep_wait();          // programmatic dependent launch, as in ffn.cu: set-up overlaps the preceding kernel's tail
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
    }
  }
  if (warp != 2) ptx::griddep_wait();
  ptx::tc_fence_before();
  __syncthreads();
  ptx::cluster_sync_all();      // the peer's barriers are initialised before anything signals them
  ptx::tc_fence_after();

  const uint32_t tmem_base = tail->tmem_base;
  const int total_tiles = tail->total_t_tiles * NB;

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
      for (int rnd = 0, tile = pair; tile < total_tiles; ++rnd, tile = tile_of(rnd, pair, num_pairs)) {
        int f_blk, t_blk;
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
        // Block-scaled variant: the tile's token scales.  A TMA box must start on a 16-byte boundary of global
        // memory (measured: a start at 4 or 8 bytes faults), i.e. on a multiple of 4 row blocks, while a tile starts
        // on any EVEN row block: fetch the aligned {4 row blocks x 32 rows} chunks that cover the tile (at most 2)
        // and point the MMA (rb0 & 3) = 0 or 2 columns into them (measured: the scale-factor TMEM address of the
        // MMA and the destination of tcgen05.cp must be even columns -- an odd one raises "misaligned address").
        const int rb0 = row0 >> 5;
        const int sf_chunks = ((rb0 & 3) + ((half + 15) >> 4) + 3) >> 2;
        const uint32_t tx_bytes = 2u * ((uint32_t)A_BYTES + (uint32_t)(narrow ? NARROW_ROWS * BK : (kMx ? B_BYTES_MX : B_BYTES)) +
                                        (kMx ? 512u + 512u * (uint32_t)sf_chunks : 0u));
        for (int kb = 0; kb < KB; ++kb) {
          ptx::mbar_wait(ptx::smem_u32(&tail->empty[stage]), phase ^ 1u);
          if (ptx::elect_one()) {
            if (rank == 0) ptx::mbar_arrive_expect_tx(ptx::smem_u32(&tail->full[stage]), tx_bytes);
            const uint32_t full = full0 + (uint32_t)stage * 8u;
            const uint32_t a_s = smem_base + (uint32_t)stage * STAGE_BYTES;
            const uint32_t b_s = a_s + A_BYTES;
            const int k0 = kb * BK;
            if (kGateUp) {
              ptx::tma_load_3d_2sm(a_s, &tmW0, full, k0, n0, e, pol_w);                 // gate -> lanes 0..63
              ptx::tma_load_3d_2sm(a_s + ATOM_BYTES, &tmW1, full, k0, n0, e, pol_w);    // up   -> lanes 64..127
            } else {
              ptx::tma_load_3d_2sm(a_s, &tmW0, full, k0, n0, e, pol_w);
              ptx::tma_load_3d_2sm(a_s + ATOM_BYTES, &tmW0, full, k0, n0 + 64, e, pol_w);
            }
            ptx::tma_load_2d_2sm(b_s, tm_b, full, k0, row_b, pol_act);
            if (kMx) {
              const int wchunk = (e * KB + kb) * mx.wchunks + n0 / FC;
              ptx::tma_load_2d_2sm(a_s + SFA_OFF, &mx.tmSFW, full, 0, wchunk, pol_w);
              for (int c = 0; c < sf_chunks; ++c)
                ptx::tma_load_3d_2sm(a_s + SFB_OFF + c * 512, &mx.tmSFB, full, (rb0 & ~3) + 4 * c, 0, kb, pol_act);
            }
          }
          __syncwarp();
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ================================================================ UMMA issuer (leader CTA)
    // The whole warp runs the loop; one elected lane issues the MMAs and the commits (always the
    // same lane: tcgen05.commit tracks the MMAs of the issuing thread).
    if (rank == 0) {
      constexpr uint32_t idesc0 = kMx ? ptx::make_idesc_mxe4m3(256, 0) : ptx::make_idesc_e4m3_f32(256, 0);
      const uint32_t sfa_t = tmem_base + SF_TMEM_COL, sfb_t = tmem_base + SF_TMEM_COL + 4;
      // descriptor = constant high word | low word (start address >> 4 in bits [0,14), LBO in [16,30))
      constexpr uint32_t DESC_HI = (1024u >> 4) | (1u << 14) | (2u << 29);
      const uint32_t smem_base = ptx::smem_u32(smem);
      const uint32_t a_lo0 = ((smem_base >> 4) & 0x3fffu) | ((16u >> 4) << 16);
      const uint32_t b_lo0 = (((smem_base + A_BYTES) >> 4) & 0x3fffu) | ((16u >> 4) << 16);
      TileCursor cur;
      int stage = 0;
      uint32_t phase = 0;
      int it = 0;
      for (int rnd = 0, tile = pair; tile < total_tiles; ++rnd, ++it, tile = tile_of(rnd, pair, num_pairs)) {
        int f_blk, t_blk;
        cur.decode(tail, tile, NB, f_blk, t_blk);
        const int e = cur.e;
        const int tsz = tail->tsz[e];
        const int row0 = tail->off[e] + t_blk * tsz;
        const int n_rows = min(tsz, tail->off[e + 1] - row0);
        const uint32_t n_mma = (uint32_t)((n_rows + 15) >> 4) << 4;
        const uint32_t sf_shift = (uint32_t)(row0 >> 5) & 3u;                    // columns into the aligned scale chunks
        const int sf_chunks = (int)((sf_shift + ((n_mma + 31) >> 5) + 3) >> 2);
        const uint32_t idesc = idesc0 | ((n_mma >> 3) << 17);
        const int acc = it & 1;
        const uint32_t acc_phase = (uint32_t)(it >> 1) & 1u;
        ptx::mbar_wait(ptx::smem_u32(&tail->tempty[acc]), acc_phase ^ 1u);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)acc * TNk;
        for (int kb = 0; kb < KB; ++kb) {
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
            // A and B: K-major SW128 -> 32 one-byte elements = 32 bytes inside the 128-byte row (+2 in units of 16 B)
            const uint32_t a_lo = a_lo0 + (uint32_t)stage * (STAGE_BYTES >> 4);
            const uint32_t b_lo = b_lo0 + (uint32_t)stage * (STAGE_BYTES >> 4);
#pragma unroll
            for (int k = 0; k < BK / UMMA_K; ++k) {
              const uint64_t da = ((uint64_t)DESC_HI << 32) | (uint64_t)(a_lo + (uint32_t)k * (UMMA_K / 16));
              const uint64_t db = ((uint64_t)DESC_HI << 32) | (uint64_t)(b_lo + (uint32_t)k * (UMMA_K / 16));
              if (kMx)
                ptx::umma_mxf8_2sm(d_tmem, da, db, idesc | ((uint32_t)k << 29) | ((uint32_t)k << 4),
                                   (uint32_t)((kb | k) != 0), sfa_t, sfb_t + sf_shift);
              else
                ptx::umma_f8_2sm(d_tmem, da, db, idesc, (uint32_t)((kb | k) != 0));
            }
            ptx::umma_commit_2sm_mc(ptx::smem_u32(&tail->empty[stage]), 3);   // frees the stage in both CTAs
            if (kb == KB - 1)
              ptx::umma_commit_2sm_mc(ptx::smem_u32(&tail->tfull[acc]), 3);   // accumulator ready in both CTAs
          }
          __syncwarp();
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else {
    // ================================================================ epilogue (warps 2..5, both CTAs)
    const int q = warp & 3;  // TMEM lane quarter this warp may access
    const int blk_par = (warp - 2) >> 2;   // down projection: which 32-column blocks (even / odd) are mine
    TileCursor cur;
    int it = 0;
    for (int rnd = 0, tile = pair; tile < total_tiles; ++rnd, ++it, tile = tile_of(rnd, pair, num_pairs)) {
      int f_blk, t_blk;
      cur.decode(tail, tile, NB, f_blk, t_blk);
      const int e = cur.e;
      const int tsz = tail->tsz[e];
      const int row0 = tail->off[e] + t_blk * tsz;
      const int n_rows = min(tsz, tail->off[e + 1] - row0);
      const int acc = it & 1;
      const uint32_t acc_phase = (uint32_t)(it >> 1) & 1u;
      // GEMM-1: the tile's row scales sx go to this warp's slice while the MMAs of the tile still run
      float* sx = sx_all + (warp - 2) * TN;
      if (kGateUp && !kMx) {
        __syncwarp();                       // the previous tile's reads of the slice are done
#pragma unroll
        for (int b = 0; b < TN / 32; ++b) {
          const int c = b * 32 + lane;
          sx[c] = (c < n_rows) ? __ldg(row_scale + row0 + c) : 0.0f;
        }
        __syncwarp();
      }
      const float se0 = kMx ? 1.0f : __ldg(sw0 + e);
      const float se1 = (kGateUp && !kMx) ? __ldg(sw1 + e) : 0.0f;
      const float she = kMx ? 1.0f : __ldg(h_scale + e);
      ptx::mbar_wait(ptx::smem_u32(&tail->tfull[acc]), acc_phase);
      ptx::tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)acc * TNk;
      if (kGateUp) {
        // lanes 0..63 gate (q = 0,1), lanes 64..127 up (q = 2,3) of the same 64 features.
        // Per 64 columns: the gate warp finishes columns 0..31 (needs the partner's up block),
        // the up warp finishes columns 32..63 (needs the partner's gate block).
        const bool is_up = q >= 2;
        const int feat = f_blk * FB + (int)rank * FC + (q & 1) * 32 + lane;
        const bool feat_ok = feat < n_total;
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
          float h[32];
          const int cbase = c0 + (is_up ? 32 : 0);
          if (kMx) {
            // the block scales were applied by the tensor core: the accumulators ARE g and u
#pragma unroll
            for (int i = 0; i < 32; ++i) {
              const float o = theirs[i * 32 + lane];
              h[i] = swiglu(is_up ? o : __uint_as_float(a[i]), is_up ? __uint_as_float(b[i]) : o);
            }
          } else {
            const float inv_sh = 1.0f / she;
#pragma unroll
            for (int i = 0; i < 32; ++i) {
              const float o = theirs[i * 32 + lane];
              const float sxi = sx[cbase + i];
              const float g = (is_up ? o : __uint_as_float(a[i])) * (sxi * se0);
              const float u = (is_up ? __uint_as_float(b[i]) : o) * (sxi * se1);
              h[i] = swiglu(g, u) * inv_sh;
            }
          }
          ptx::named_bar_sync(bar_id, 64);     // both blocks consumed before the next publish
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
            const int fb = feat >> 5;      // warp-uniform: (f_blk * FB + rank * FC + (q & 1) * 32) / 32
            if (feat_ok && cbase + lane < n_rows)
              mx.hsf[((size_t)((fb >> 2) * 32 + (r & 31)) * (size_t)mx.Rb + (size_t)(r >> 5)) * 4 + (size_t)(fb & 3)] = (uint8_t)my_byte;
          }
          store_block_T_e4m3(h, reinterpret_cast<uint8_t*>(out_v), (size_t)ld_out, row0 + cbase, n_rows - cbase, feat,
                             feat_ok, lane);
        }
      } else {
        const int feat = f_blk * FB + (int)rank * FC + q * 32 + lane;
        const bool feat_ok = feat < n_total;
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
          for (int i = 0; i < 32; ++i) v[i] = kMx ? __uint_as_float(a[i]) : __uint_as_float(a[i]) * (she * se0);
          store_block_T(v, reinterpret_cast<__nv_bfloat16*>(out_v), (size_t)ld_out, row0 + c0, n_rows - c0, feat, feat_ok,
                        lane);
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
// lifetime, keyed by (pointer, shape): weights and workspaces are long-lived in serving.
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

struct MapKey {
  const void* ptr;
  uint64_t d0, d1, d2;
  uint32_t b0, b1;
  bool words;
  bool operator==(const MapKey& o) const {
    return ptr == o.ptr && d0 == o.d0 && d1 == o.d1 && d2 == o.d2 && b0 == o.b0 && b1 == o.b1 && words == o.words;
  }
};
struct MapKeyHash {
  size_t operator()(const MapKey& k) const {
    size_t h = reinterpret_cast<size_t>(k.ptr);
    h = h * 1315423911u ^ k.d0;
    h = h * 1315423911u ^ k.d1;
    h = h * 1315423911u ^ k.d2;
    h = h * 1315423911u ^ ((uint64_t)k.b0 << 32 | k.b1);
    h = h * 1315423911u ^ (k.words ? 1u : 0u);
    return h;
  }
};
std::mutex g_map_mu;
std::unordered_map<MapKey, CUtensorMap, MapKeyHash> g_maps;

// rank 2: dims (d0 inner, d1); rank 3: dims (d0 inner, d1, d2).  One-byte elements, 128-byte swizzle --
// or (words) 32-bit elements without swizzle: the scale-factor arrays of the block-scaled variant.
vibe_status get_tensor_map(const void* ptr, uint64_t d0, uint64_t d1, uint64_t d2, uint32_t box0, uint32_t box1,
                           CUtensorMap* out, bool words = false) {
  MapKey key{ptr, d0, d1, d2, box0, box1, words};
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
  cuuint64_t dims[3] = {d0, d1, r3 ? d2 : 1};
  const uint64_t esz = words ? 4 : 1;
  cuuint64_t strides[2] = {d0 * esz, d0 * d1 * esz};
  cuuint32_t box[3] = {box0, box1, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUtensorMap m;
  CUresult r = enc(&m, words ? CU_TENSOR_MAP_DATA_TYPE_UINT32 : CU_TENSOR_MAP_DATA_TYPE_UINT8, r3 ? 3 : 2,
                   const_cast<void*>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   words ? CU_TENSOR_MAP_SWIZZLE_NONE : CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
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

// the opt-in to > 48 KB of dynamic shared memory is per device: done once for each device this process uses
vibe_status set_smem_attrs() {
  static std::mutex mu;
  static bool done[kMaxDevices] = {};
  const int dev = current_device();
  std::lock_guard<std::mutex> lk(mu);
  if (done[dev]) return VIBE_OK;
  VIBE_CUDA(cudaFuncSetAttribute(ffn8_gemm_kernel<0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES));
  VIBE_CUDA(cudaFuncSetAttribute(ffn8_gemm_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES));
  VIBE_CUDA(cudaFuncSetAttribute(ffn8_gemm_kernel<0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES));
  VIBE_CUDA(cudaFuncSetAttribute(ffn8_gemm_kernel<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES));
  done[dev] = true;
  return VIBE_OK;
}

}  // namespace

vibe_status grouped_ffn_fp8_impl(const void* Xq, const float* row_scale, const int32_t* offsets, int E_loc, int R_cap,
                                 int d, int f, const void* W1q, const float* s1, const void* W3q, const float* s3,
                                 const void* W2q, const float* s2, const float* h_scale, void* Hq, void* Y,
                                 cudaStream_t st) {
  CUtensorMap tmX, tmH, tmXN, tmHN, tmW1, tmW3, tmW2;
  vibe_status s;
  // activations [R_cap, K] and packed weights [E_loc, N, K]: K innermost, boxes of 128 K x (128 | 32 | 64) rows
  if ((s = get_tensor_map(Xq, d, R_cap, 0, BK, TN / 2, &tmX)) != VIBE_OK) return s;
  if ((s = get_tensor_map(Hq, f, R_cap, 0, BK, TN / 2, &tmH)) != VIBE_OK) return s;
  if ((s = get_tensor_map(Xq, d, R_cap, 0, BK, NARROW_ROWS, &tmXN)) != VIBE_OK) return s;
  if ((s = get_tensor_map(Hq, f, R_cap, 0, BK, NARROW_ROWS, &tmHN)) != VIBE_OK) return s;
  if ((s = get_tensor_map(W1q, d, f, E_loc, BK, 64, &tmW1)) != VIBE_OK) return s;
  if ((s = get_tensor_map(W3q, d, f, E_loc, BK, 64, &tmW3)) != VIBE_OK) return s;
  if ((s = get_tensor_map(W2q, f, d, E_loc, BK, 64, &tmW2)) != VIBE_OK) return s;
  vibe_status sa = set_smem_attrs();
  if (sa != VIBE_OK) return sa;
  const int grid = num_sms() & ~1;   // CTA pairs (clusters of 2)
  const float* none = nullptr;
  const MxArgs no_mx{};
  cudaError_t le = launch_pdl(ffn8_gemm_kernel<0, false>, dim3(grid), dim3(num_threads(0)), SMEM_BYTES, st, tmX, tmXN, tmW1, tmW3,
                              offsets, E_loc, f, d, Hq, f, row_scale, s1, s3, h_scale, no_mx);
  VIBE_REQUIRE(le == cudaSuccess, VIBE_ERR_CUDA, "ffn8_gemm_kernel<gate_up> launch failed: %s", cudaGetErrorString(le));
  VIBE_LAUNCH_CHECK("ffn8_gemm_kernel<gate_up>");
  le = launch_pdl(ffn8_gemm_kernel<1, false>, dim3(grid), dim3(num_threads(1)), SMEM_BYTES, st, tmH, tmHN, tmW2, tmW2, offsets,
                  E_loc, d, f, Y, d, none, s2, none, h_scale, no_mx);
  VIBE_REQUIRE(le == cudaSuccess, VIBE_ERR_CUDA, "ffn8_gemm_kernel<down> launch failed: %s", cudaGetErrorString(le));
  VIBE_LAUNCH_CHECK("ffn8_gemm_kernel<down>");
  return VIBE_OK;
}

// Block-scaled variant.  sf13: joint gate|up weight scales (one 512-byte chunk per expert, K stage and 64 features:
// TMEM rows 0..63 = W1's, 64..127 = W3's); sf2: down-projection weight scales (chunk per 128 features); xsf / hsf:
// token scales [K/128][32][Rb] words (hsf is written by GEMM-1 and read by GEMM-2).
vibe_status grouped_ffn_mxfp8_impl(const void* Xq, const void* xsf, const int32_t* offsets, int E_loc, int R_cap, int d,
                                   int f, const void* W1q, const void* W3q, const void* sf13, const void* W2q,
                                   const void* sf2, void* Hq, void* hsf, void* Y, cudaStream_t st) {
  CUtensorMap tmX, tmH, tmXN, tmHN, tmW1, tmW3, tmW2;
  MxArgs m1{}, m2{};
  vibe_status s;
  const int Rb = mx_row_blocks(R_cap);
  if ((s = get_tensor_map(Xq, d, R_cap, 0, BK, TN_MX / 2, &tmX)) != VIBE_OK) return s;
  if ((s = get_tensor_map(Hq, f, R_cap, 0, BK, TN_MX / 2, &tmH)) != VIBE_OK) return s;
  if ((s = get_tensor_map(Xq, d, R_cap, 0, BK, NARROW_ROWS, &tmXN)) != VIBE_OK) return s;
  if ((s = get_tensor_map(Hq, f, R_cap, 0, BK, NARROW_ROWS, &tmHN)) != VIBE_OK) return s;
  if ((s = get_tensor_map(W1q, d, f, E_loc, BK, 64, &tmW1)) != VIBE_OK) return s;
  if ((s = get_tensor_map(W3q, d, f, E_loc, BK, 64, &tmW3)) != VIBE_OK) return s;
  if ((s = get_tensor_map(W2q, f, d, E_loc, BK, 64, &tmW2)) != VIBE_OK) return s;
  m1.wchunks = f / 64;
  m2.wchunks = d / 128;
  if ((s = get_tensor_map(sf13, 128, (uint64_t)E_loc * (d / BK) * m1.wchunks, 0, 128, 1, &m1.tmSFW, true)) != VIBE_OK) return s;
  if ((s = get_tensor_map(sf2, 128, (uint64_t)E_loc * (f / BK) * m2.wchunks, 0, 128, 1, &m2.tmSFW, true)) != VIBE_OK) return s;
  if ((s = get_tensor_map(xsf, Rb, 32, d / BK, 4, 32, &m1.tmSFB, true)) != VIBE_OK) return s;
  if ((s = get_tensor_map(hsf, Rb, 32, f / BK, 4, 32, &m2.tmSFB, true)) != VIBE_OK) return s;
  m1.hsf = reinterpret_cast<uint8_t*>(hsf);
  m1.Rb = m2.Rb = Rb;
  vibe_status sa = set_smem_attrs();
  if (sa != VIBE_OK) return sa;
  const int grid = num_sms() & ~1;
  const float* none = nullptr;
  cudaError_t le = launch_pdl(ffn8_gemm_kernel<0, true>, dim3(grid), dim3(num_threads(0)), SMEM_BYTES, st, tmX, tmXN, tmW1,
                              tmW3, offsets, E_loc, f, d, Hq, f, none, none, none, none, m1);
  VIBE_REQUIRE(le == cudaSuccess, VIBE_ERR_CUDA, "ffn8_gemm_kernel<gate_up, mx> launch failed: %s", cudaGetErrorString(le));
  VIBE_LAUNCH_CHECK("ffn8_gemm_kernel<gate_up, mx>");
  le = launch_pdl(ffn8_gemm_kernel<1, true>, dim3(grid), dim3(num_threads(1)), SMEM_BYTES, st, tmH, tmHN, tmW2, tmW2,
                  offsets, E_loc, d, f, Y, d, none, none, none, none, m2);
  VIBE_REQUIRE(le == cudaSuccess, VIBE_ERR_CUDA, "ffn8_gemm_kernel<down, mx> launch failed: %s", cudaGetErrorString(le));
  VIBE_LAUNCH_CHECK("ffn8_gemm_kernel<down, mx>");
  return VIBE_OK;
}

}  // namespace vibe

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
                              reinterpret_cast<cudaStream_t>(stream));
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
                                reinterpret_cast<cudaStream_t>(stream));
}
