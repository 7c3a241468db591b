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
// Semantics: include/vibe.h (vibe_grouped_ffn); F1-F4.
#include <mutex>
#include <unordered_map>
#include <string>
#include <cstring>

#include "common.cuh"
#include "ptx.cuh"

namespace vibe {
namespace {

constexpr int BK = 64;                  // K per smem stage (one 128-byte swizzle atom of bf16)
constexpr int TN = 256;                 // tokens per tile = max UMMA N
constexpr int UMMA_K = 16;
constexpr int STAGES = 6;
constexpr int ATOM_BYTES = 64 * BK * 2;         // 8 KB : 64 features x 64 K (MN-major, SW128)
constexpr int A_BYTES = 2 * ATOM_BYTES;         // 16 KB: this CTA's 128 accumulator lanes
constexpr int B_BYTES = (TN / 2) * BK * 2;      // 16 KB: this CTA's half of the token tile
constexpr int STAGE_BYTES = A_BYTES + B_BYTES;  // 32 KB
constexpr int NARROW_ROWS = 32;                 // rows of the small activation box (per CTA)
constexpr int XCHG_BYTES = 16384;               // gate/up swap: 2 warp pairs x 2 directions x 4 KB
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
constexpr size_t SPLIT_WS_BYTES = SPLIT_PART_BYTES + 2 * (size_t)SPLIT_COUNTERS * sizeof(int);   // counters of GEMM-1, of GEMM-2

struct SmemTail {
  uint64_t full[STAGES];          // leader CTA: both CTAs' TMA bytes of a stage have landed
  uint64_t empty[STAGES];         // each CTA: the MMAs reading the stage have retired
  uint64_t tfull[2];              // each CTA: accumulator stage complete
  uint64_t tempty[2];             // leader CTA: all 8 epilogue warps of the pair drained it
  uint32_t tmem_base;
  int32_t total_t_tiles;
  int32_t split;                  // K slices of a split tile (1 = no split-K)
  int32_t split_from;             // first split tile: tiles [split_from, total) are cut into `split` K slices
  int32_t off[MAX_SLOTS + 1];     // segment starts (rows)
  int32_t cum[MAX_SLOTS + 1];     // exclusive prefix of token tiles per slot
  int32_t tsz[MAX_SLOTS];         // rows per token tile of the slot (multiple of 16, <= TN)
};
constexpr size_t SMEM_BYTES = 1024 + (size_t)STAGES * STAGE_BYTES + XCHG_BYTES + sizeof(SmemTail);
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

// kMode: 0 = gate|up + SwiGLU (GEMM-1), 1 = down (GEMM-2), 2 = down with the gate-weighted
// scatter fused into the epilogue (vibe_grouped_ffn_scatter).
template <int kMode>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(num_threads(kMode), 1)
ffn_gemm_kernel(const __grid_constant__ CUtensorMap tmAct, const __grid_constant__ CUtensorMap tmActN,
                const __grid_constant__ CUtensorMap tmW0, const __grid_constant__ CUtensorMap tmW1, const int32_t* __restrict__ offsets, int E_loc,
                int n_total, int k_total, __nv_bfloat16* __restrict__ out, int ld_out,
                const int32_t* __restrict__ row_to_assign, const float* __restrict__ topk_w,
                float* __restrict__ split_part /*NULL: no split-K*/, int* __restrict__ split_cnt) {
  constexpr bool kGateUp = (kMode == 0);
  constexpr int FB = kGateUp ? 128 : 256;   // output features per pair tile
  constexpr int FC = FB / 2;                // ... per CTA
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  float* xchg = reinterpret_cast<float*>(smem + (size_t)STAGES * STAGE_BYTES);
  SmemTail* tail = reinterpret_cast<SmemTail*>(smem + (size_t)STAGES * STAGE_BYTES + XCHG_BYTES);
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
      const int nt = (hi - lo + TN - 1) / TN;
      if (e < E_loc) tail->tsz[e] = nt > 0 ? ((((hi - lo + nt - 1) / nt) + 15) & ~15) : TN;
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
      for (int rnd = 0, unit = pair; unit < total_units; ++rnd, unit = tile_of(rnd, pair, num_pairs)) {
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
        const uint32_t tx_bytes = narrow ? 2u * (A_BYTES + NARROW_ROWS * BK * 2) : 2u * STAGE_BYTES;
        for (int kb = kb_lo; kb < kb_hi; ++kb) {
          ptx::mbar_wait(ptx::smem_u32(&tail->empty[stage]), phase ^ 1u);
          if (ptx::elect_one()) {
            if (rank == 0) ptx::mbar_arrive_expect_tx(ptx::smem_u32(&tail->full[stage]), tx_bytes);
            const uint32_t full = full0 + (uint32_t)stage * 8u;
            const uint32_t a_s = smem_base + (uint32_t)stage * STAGE_BYTES;
            const uint32_t b_s = a_s + A_BYTES;
            const int k0 = kb * BK;
            if (kGateUp) {
              ptx::tma_load_3d_2sm(a_s, &tmW0, full, n0, k0, e, pol_w);                 // gate -> lanes 0..63
              ptx::tma_load_3d_2sm(a_s + ATOM_BYTES, &tmW1, full, n0, k0, e, pol_w);    // up   -> lanes 64..127
            } else {
              ptx::tma_load_3d_2sm(a_s, &tmW0, full, n0, k0, e, pol_w);
              ptx::tma_load_3d_2sm(a_s + ATOM_BYTES, &tmW0, full, n0 + 64, k0, e, pol_w);
            }
            ptx::tma_load_2d_2sm(b_s, tm_b, full, k0, row_b, pol_act);
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
      constexpr uint32_t idesc0 = ptx::make_idesc_bf16_f32(256, 0, /*a_mn=*/true, /*b_mn=*/false);
      // descriptor = constant high word | low word (start address >> 4 in bits [0,14), LBO in [16,30))
      constexpr uint32_t DESC_HI = (1024u >> 4) | (1u << 14) | (2u << 29);
      const uint32_t smem_base = ptx::smem_u32(smem);
      const uint32_t a_lo0 = ((smem_base >> 4) & 0x3fffu) | ((uint32_t)(ATOM_BYTES >> 4) << 16);
      const uint32_t b_lo0 = (((smem_base + A_BYTES) >> 4) & 0x3fffu) | ((16u >> 4) << 16);
      TileCursor cur;
      int stage = 0;
      uint32_t phase = 0;
      int it = 0;
      for (int rnd = 0, unit = pair; unit < total_units; ++rnd, ++it, unit = tile_of(rnd, pair, num_pairs)) {
        int f_blk, t_blk;
        const bool is_split = unit >= split_from;
        const int tile = is_split ? split_from + (unit - split_from) / S : unit;
        const int slice = is_split ? (unit - split_from) % S : 0, nsl = is_split ? S : 1;
        const int kb_lo = slice * KB / nsl, kb_hi = (slice + 1) * KB / nsl;
        cur.decode(tail, tile, NB, f_blk, t_blk);
        const int e = cur.e;
        const int tsz = tail->tsz[e];
        const int n_rows = min(tsz, tail->off[e + 1] - (tail->off[e] + t_blk * tsz));
        const uint32_t n_mma = (uint32_t)((n_rows + 15) >> 4) << 4;
        const uint32_t idesc = idesc0 | ((n_mma >> 3) << 17);
        const int acc = it & 1;
        const uint32_t acc_phase = (uint32_t)(it >> 1) & 1u;
        ptx::mbar_wait(ptx::smem_u32(&tail->tempty[acc]), acc_phase ^ 1u);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)acc * TN;
        for (int kb = kb_lo; kb < kb_hi; ++kb) {
          ptx::mbar_wait(ptx::smem_u32(&tail->full[stage]), phase);
          ptx::tc_fence_after();
          if (ptx::elect_one()) {
            // A: MN-major SW128 -> 16 K-rows = 2 swizzle atoms of 1024 B (+128 in units of 16 B);
            // B: K-major SW128 -> 16 elements = 32 bytes inside the 128-byte row (+2)
            const uint32_t a_lo = a_lo0 + (uint32_t)stage * (STAGE_BYTES >> 4);
            const uint32_t b_lo = b_lo0 + (uint32_t)stage * (STAGE_BYTES >> 4);
#pragma unroll
            for (int k = 0; k < BK / UMMA_K; ++k) {
              const uint64_t da = ((uint64_t)DESC_HI << 32) | (uint64_t)(a_lo + (uint32_t)k * (UMMA_K * 128 / 16));
              const uint64_t db = ((uint64_t)DESC_HI << 32) | (uint64_t)(b_lo + (uint32_t)k * (UMMA_K * 2 / 16));
              ptx::umma_bf16_2sm(d_tmem, da, db, idesc, (uint32_t)((kb > kb_lo) | (k != 0)));
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
  } else {
    // ================================================================ epilogue (warps 2..5, both CTAs)
    const int q = warp & 3;  // TMEM lane quarter this warp may access
    const int blk_par = (warp - 2) >> 2;   // down projection: which 32-column blocks (even / odd) are mine
    TileCursor cur;
    int it = 0;
    for (int rnd = 0, unit = pair; unit < total_units; ++rnd, ++it, unit = tile_of(rnd, pair, num_pairs)) {
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
      ptx::mbar_wait(ptx::smem_u32(&tail->tfull[acc]), acc_phase);
      ptx::tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)acc * TN;
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
            const int feat = f_blk * FB + (int)rank * FC + (q & 1) * 32 + lane;
            const bool feat_ok = feat < n_total;
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
              for (int i = 0; i < 32; ++i) g[i] = swiglu(g[i], u[i]);
              store_block_T(g, out, (size_t)ld_out, row0 + c0, n_rows - c0, feat, feat_ok, lane);
            }
          } else {
            const int feat = f_blk * FB + (int)rank * FC + q * 32 + lane;
            const bool feat_ok = feat < n_total;
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
              if (kMode == 2)
                store_block_T_scatter(v, out, (size_t)ld_out, feat, feat_ok, lane, sc_wt + c0, sc_asg + c0);
              else
                store_block_T(v, out, (size_t)ld_out, row0 + c0, n_rows - c0, feat, feat_ok, lane);
            }
          }
        }
        continue;
      }
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
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            const float o = theirs[i * 32 + lane];
            h[i] = is_up ? swiglu(o, __uint_as_float(b[i])) : swiglu(__uint_as_float(a[i]), o);
          }
          ptx::named_bar_sync(bar_id, 64);     // both blocks consumed before the next publish
          const int cbase = c0 + (is_up ? 32 : 0);
          store_block_T(h, out, (size_t)ld_out, row0 + cbase, n_rows - cbase, feat, feat_ok, lane);
        }
      } else {
        const int feat = f_blk * FB + (int)rank * FC + q * 32 + lane;
        const bool feat_ok = feat < n_total;
#pragma unroll
        for (int b = 0; b < TN / 32; ++b) {
          const int c0 = b * 32;
          if (c0 >= n_rows) break;
          if ((b & 1) != blk_par) continue;
          uint32_t a[32];
          ptx::tmem_ld_32x32(taddr + c0, a);
          ptx::tmem_ld_wait();
          float v[32];
#pragma unroll
          for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(a[i]);
          if (kMode == 2)
            store_block_T_scatter(v, out, (size_t)ld_out, feat, feat_ok, lane, sc_wt + c0, sc_asg + c0);
          else
            store_block_T(v, out, (size_t)ld_out, row0 + c0, n_rows - c0, feat, feat_ok, lane);
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
  bool operator==(const MapKey& o) const {
    return ptr == o.ptr && d0 == o.d0 && d1 == o.d1 && d2 == o.d2 && b0 == o.b0 && b1 == o.b1;
  }
};
struct MapKeyHash {
  size_t operator()(const MapKey& k) const {
    size_t h = reinterpret_cast<size_t>(k.ptr);
    h = h * 1315423911u ^ k.d0;
    h = h * 1315423911u ^ k.d1;
    h = h * 1315423911u ^ k.d2;
    h = h * 1315423911u ^ ((uint64_t)k.b0 << 32 | k.b1);
    return h;
  }
};
std::mutex g_map_mu;
std::unordered_map<MapKey, CUtensorMap, MapKeyHash> g_maps;

// rank 2: dims (d0 inner, d1); rank 3: dims (d0 inner, d1, d2).  bf16, 128-byte swizzle.
vibe_status get_tensor_map(const void* ptr, uint64_t d0, uint64_t d1, uint64_t d2, uint32_t box0, uint32_t box1,
                           CUtensorMap* out) {
  MapKey key{ptr, d0, d1, d2, box0, box1};
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
  cuuint64_t strides[2] = {d0 * 2, d0 * d1 * 2};
  cuuint32_t box[3] = {box0, box1, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUtensorMap m;
  CUresult r = enc(&m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, r3 ? 3 : 2, const_cast<void*>(ptr), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
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

}  // namespace

size_t grouped_ffn_ws_bytes() { return SPLIT_WS_BYTES; }
vibe_status grouped_ffn_zero_counters(void* ws, cudaStream_t st) {
  VIBE_CUDA(cudaMemsetAsync(reinterpret_cast<char*>(ws) + SPLIT_PART_BYTES, 0, 2 * (size_t)SPLIT_COUNTERS * sizeof(int), st));
  return VIBE_OK;
}

// ws (may be NULL or short: split-K is then off): SPLIT_WS_BYTES bytes; ws_zeroed: the caller has already zeroed the
// counters behind the partial buffer on this stream (the layer entry does it before the route kernel so that no
// memset sits between the permutation and the FFN kernels, which are chained by programmatic dependent launch)
vibe_status grouped_ffn_impl(const void* Xp, const int32_t* offsets, int E_loc, int R_cap, int d, int f,
                             const void* W1, const void* W3, const void* W2, void* H_ws, void* Y,
                             cudaStream_t st, const int32_t* row_to_assign, const float* topk_w, void* ws,
                             size_t ws_bytes, bool ws_zeroed) {
  CUtensorMap tmX, tmH, tmXN, tmHN, tmW1, tmW3, tmW2;
  vibe_status s;
  if ((s = get_tensor_map(Xp, d, R_cap, 0, BK, TN / 2, &tmX)) != VIBE_OK) return s;
  if ((s = get_tensor_map(H_ws, f, R_cap, 0, BK, TN / 2, &tmH)) != VIBE_OK) return s;
  if ((s = get_tensor_map(Xp, d, R_cap, 0, BK, NARROW_ROWS, &tmXN)) != VIBE_OK) return s;
  if ((s = get_tensor_map(H_ws, f, R_cap, 0, BK, NARROW_ROWS, &tmHN)) != VIBE_OK) return s;
  if ((s = get_tensor_map(W1, f, d, E_loc, 64, BK, &tmW1)) != VIBE_OK) return s;
  if ((s = get_tensor_map(W3, f, d, E_loc, 64, BK, &tmW3)) != VIBE_OK) return s;
  if ((s = get_tensor_map(W2, d, f, E_loc, 64, BK, &tmW2)) != VIBE_OK) return s;
  {
    // the opt-in to > 48 KB of dynamic shared memory is per device: once for each device this process uses
    static std::mutex mu;
    static bool done[kMaxDevices] = {};
    const int dev = current_device();
    std::lock_guard<std::mutex> lk(mu);
    if (!done[dev]) {
      VIBE_CUDA(cudaFuncSetAttribute(ffn_gemm_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES));
      VIBE_CUDA(cudaFuncSetAttribute(ffn_gemm_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES));
      VIBE_CUDA(cudaFuncSetAttribute(ffn_gemm_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES));
      done[dev] = true;
    }
  }
  const int grid = num_sms() & ~1;   // CTA pairs (clusters of 2)
  // both launches carry the programmatic-dependent-launch attribute (see the kernel's set-up)
  const int32_t* no_map = nullptr;
  const float* no_w = nullptr;
  float* part = nullptr;
  int* cnt1 = nullptr;
  int* cnt2 = nullptr;
  if (ws != nullptr && ws_bytes >= SPLIT_WS_BYTES && (reinterpret_cast<uintptr_t>(ws) & 15u) == 0) {
    part = reinterpret_cast<float*>(ws);
    cnt1 = reinterpret_cast<int*>(reinterpret_cast<char*>(ws) + SPLIT_PART_BYTES);
    cnt2 = cnt1 + SPLIT_COUNTERS;
    if (!ws_zeroed) VIBE_CUDA(cudaMemsetAsync(cnt1, 0, 2 * (size_t)SPLIT_COUNTERS * sizeof(int), st));
  }
  cudaError_t le = launch_pdl(ffn_gemm_kernel<0>, dim3(grid), dim3(num_threads(0)), SMEM_BYTES, st, tmX, tmXN, tmW1, tmW3,
                              offsets, E_loc, f, d, reinterpret_cast<__nv_bfloat16*>(H_ws), f, no_map, no_w, part, cnt1);
  VIBE_REQUIRE(le == cudaSuccess, VIBE_ERR_CUDA, "ffn_gemm_kernel<gate_up> launch failed: %s", cudaGetErrorString(le));
  VIBE_LAUNCH_CHECK("ffn_gemm_kernel<gate_up>");
  if (row_to_assign != nullptr)
    le = launch_pdl(ffn_gemm_kernel<2>, dim3(grid), dim3(num_threads(2)), SMEM_BYTES, st, tmH, tmHN, tmW2, tmW2, offsets,
                    E_loc, d, f, reinterpret_cast<__nv_bfloat16*>(Y), d, row_to_assign, topk_w, part, cnt2);
  else
    le = launch_pdl(ffn_gemm_kernel<1>, dim3(grid), dim3(num_threads(1)), SMEM_BYTES, st, tmH, tmHN, tmW2, tmW2, offsets,
                    E_loc, d, f, reinterpret_cast<__nv_bfloat16*>(Y), d, no_map, no_w, part, cnt2);
  VIBE_REQUIRE(le == cudaSuccess, VIBE_ERR_CUDA, "ffn_gemm_kernel<down> launch failed: %s", cudaGetErrorString(le));
  VIBE_LAUNCH_CHECK("ffn_gemm_kernel<down>");
  return VIBE_OK;
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
