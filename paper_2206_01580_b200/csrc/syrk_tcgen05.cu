// syrk_tcgen05.cu -- step a8: the normal equations ZtZ (+)= A^T A, Zty (+)= A^T y (eq. 16,
// eq. 17) on the 5th-generation tensor cores with fp32-level accuracy: every operand is split into a
// high and a low part with 11 significant bits each, the product is hi*hi + hi*lo + lo*hi (three MMAs, small
// terms first), and the row dimension is cut into 128-row chunks whose partial products are summed in fp32
// round-to-nearest (the paper's FP32 round-off remark, L351, restated for a truncating TMEM accumulator).
//
// Two operand containers (qmll_normal_equations_mode):
//   QMLL_NE_SPLIT_F16  (default)  hi/lo are fp16 (kind::f16, K = 16 per MMA).  fp16 and TF32 carry the same 11
//       significant bits, so the split is as exact as 3xTF32, but the f16 MMA runs at twice the TF32 rate and the
//       operands are half as large.  fp16's narrow exponent is handled by one power-of-two scale per
//       (128-row chunk, 128-column block), measured by the split pass and undone exactly in the epilogue.
//   QMLL_NE_SPLIT_TF32            hi/lo are TF32 in fp32 containers (kind::tf32, K = 8 per MMA): the 3xTF32 scheme.
//
// Pipeline of one call (per panel of rows that fits the workspace):
//   1. split_kernel: A[rows, D] -> At_hi, At_lo, k-block-major [R_pad/BK][D][BK] (the contraction index `row` is
//      the contiguous one inside each BK-row block, BK*elem = 128 bytes: one TMA box = 16 KB contiguous); per-block
//      partial sums of A^T y ride along and are reduced deterministically in fp64 by zty_reduce_kernel.
//   2. syrk_tcgen05_kernel: persistent, warp-specialised.  One CTA owns a 128 x 256 tile T = At[I,:] At[J,:]^T
//      for ALL rows: TMA (SWIZZLE_128B) -> 2-stage smem ring -> tcgen05.mma (lo*hi + hi*lo + hi*hi) into one of
//      two 256-column TMEM accumulators; every 128 rows the accumulator is drained by 8 epilogue warps
//      (tcgen05.ld) and summed in registers in fp32 while the next chunk is already running.  The tile is written
//      transposed (C[J0+j, I0+i], coalesced along i); only tiles touching the lower triangle are computed.
//   3. mirror_lower_kernel: C[i, j] = C[j, i] for i < j  -> full, exactly symmetric matrix.
#include <cuda.h>
#include <cuda_fp16.h>
#include <mutex>

#include "qmll_common.cuh"
#include "ptx_utils.cuh"
#include "tcgen05_utils.cuh"

namespace qmll {

constexpr int kBM = 128;          // tile extent along I (MMA M, TMEM lanes)
constexpr int kBN = 256;          // tile extent along J (MMA N, TMEM columns)
constexpr int kStages = 2;
// Rows accumulated in TMEM before a drain.  The tensor core truncates (rounds toward zero) every accumulate, a
// bias of ~2e-8 per MMA relative to the running sum, so long same-sign sums (Gram diagonals, coherent Z columns)
// need short chunks (measured: 1024 rows 1.0e-5, 128 rows 1.0e-6 relative); chunk partials are summed in fp32
// round-to-nearest.  A compile-time constant: it is part of the numerics of the call.
constexpr int kChunkRows = 128;
constexpr int kPanelRows = 1024;  // panel granularity (rows) when the workspace cannot hold all rows
constexpr long long kMaxPanelRows = 32768;  // see syrk_impl (measured: 100 000 x 16384 in 4 panels 68.7 ms, in one 85.0 ms)
constexpr int kColBlock = 128;    // column granularity of the fp16 scales and of the split pass
constexpr int kSyrkThreads = 320; // warp 0 TMA producer, warp 1 MMA issuer, warps 2..9 epilogue
constexpr uint32_t kTileABytes = kBM * 128;                 // 128 features x 128 bytes of rows: 16 KB
constexpr uint32_t kTileBBytes = kBN * 128;                 // 32 KB
constexpr uint32_t kStageBytes = 2 * kTileABytes + 2 * kTileBBytes;  // hi + lo of both operands: 96 KB
constexpr uint32_t kSmemBytes = kStages * kStageBytes + 256 + 1024;  // + barriers + alignment slack
// CTA pairs (cta_group::2): the pair computes a 256 x 256 block of C; each CTA holds its own 128 rows of the I operand
// and HALF of the J operand (128 of the 256 columns), so a stage is 64 KB per CTA and three of them fit.
constexpr int kStagesP = 3;
constexpr uint32_t kStageBytesP = 4 * kTileABytes;
constexpr uint32_t kSmemBytesP = kStagesP * kStageBytesP + 512 + 1024;

template <bool F16>
struct SplitMode {
  static constexpr int kElemBytes = F16 ? 2 : 4;
  static constexpr int kBK = 128 / kElemBytes;      // rows per pipeline stage = one 128-byte swizzle span
  static constexpr int kUmmaK = 32 / kElemBytes;    // rows per tcgen05.mma (32 bytes)
  static constexpr int kTileRows = 2 * kBK;         // rows per block of the split pass (F16: one chunk)
  static constexpr uint32_t kFmt = F16 ? 0u : 2u;   // instruction-descriptor operand format: 0 = F16, 2 = TF32
  // Instruction descriptor: D fp32, A/B as kFmt, both K-major, N = 256, M = 128.
  static constexpr uint32_t kIdesc = (1u << 4) | (kFmt << 7) | (kFmt << 10) | ((uint32_t)(kBN >> 3) << 17) |
                                     ((uint32_t)(kBM >> 4) << 24);
};

// ---------------------------------------------------------------------------------------------------
// PTX wrappers
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
      : "memory");
}
__device__ __forceinline__ float to_tf32(float a) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(a));
  return __uint_as_float(r);
}

// ---------------------------------------------------------------------------------------------------
// 1. split (+ scale) + transpose (+ partial A^T y).  Block: kTileRows rows x 128 features, 8 warps; a warp owns
//    kTileRows/8 adjacent rows, a lane the features lane, lane+32, lane+64, lane+96 of the block (coalesced 128-byte
//    loads whatever D is).  The hi/lo values of a feature for the warp's rows are 32 contiguous bytes of the output.
// ---------------------------------------------------------------------------------------------------
constexpr int kSplitColBytes = 256 + 16;  // shared-memory bytes per feature (two 128-byte k-blocks + pad: no conflicts)
constexpr int kSplitSmem = 2 * kColBlock * kSplitColBytes;

template <bool F16>
__global__ void __launch_bounds__(256)
split_kernel(const float* __restrict__ A, const float* __restrict__ y, long long rows, int D,
             uint8_t* __restrict__ At_hi, uint8_t* __restrict__ At_lo, float* __restrict__ inv_scale, int n_cb,
             float* __restrict__ zty_part) {
  using M = SplitMode<F16>;
  constexpr int RPW = M::kTileRows / 8;   // rows per warp: 16 (F16) / 8 (TF32)
  extern __shared__ __align__(16) uint8_t sm[];
  __shared__ float red[8];
  __shared__ float ysum[8][kColBlock];
  uint8_t* sm_hi = sm;
  uint8_t* sm_lo = sm + kColBlock * kSplitColBytes;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long rb = blockIdx.x;
  const int cb = blockIdx.y, c0 = cb * kColBlock;
  const long long r0 = rb * M::kTileRows + warp * RPW;

  float v[RPW][4];
  float zacc[4] = {0.f, 0.f, 0.f, 0.f};
  float amax = 0.f;
#pragma unroll
  for (int rr = 0; rr < RPW; ++rr) {
    const long long r = r0 + rr;
    const float yv = (y != nullptr && r < rows) ? __ldg(y + r) : 0.f;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const int col = c0 + lane + 32 * c;
      const float a = (r < rows && col < D) ? __ldcs(A + (size_t)r * D + col) : 0.f;
      v[rr][c] = a;
      amax = fmaxf(amax, fabsf(a));
      zacc[c] = fmaf(a, yv, zacc[c]);
    }
  }
  float s = 1.f;
  if constexpr (F16) {
    // one power-of-two scale per block: amax * s in [2^13, 2^14), undone exactly by the tcgen05 kernel's epilogue
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, m));
    if (lane == 0) red[warp] = amax;
    __syncthreads();
    amax = red[0];
#pragma unroll
    for (int w = 1; w < 8; ++w) amax = fmaxf(amax, red[w]);
    int e = (int)((__float_as_uint(amax) >> 23) & 0xffu) - 127;   // floor(log2 amax) for normal numbers
    int sh = 13 - e;
    if (amax == 0.f) sh = 0;
    sh = sh < -100 ? -100 : (sh > 100 ? 100 : sh);
    s = __uint_as_float((uint32_t)(127 + sh) << 23);
    if (threadIdx.x == 0) inv_scale[rb * n_cb + cb] = __uint_as_float((uint32_t)(127 - sh) << 23);
  }
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const int cl = lane + 32 * c;
    uint4 h[2], l[2];
    if constexpr (F16) {
      __half hh[RPW], ll[RPW];
#pragma unroll
      for (int rr = 0; rr < RPW; ++rr) {
        const float a = v[rr][c] * s;
        hh[rr] = __float2half_rn(a);
        ll[rr] = __float2half_rn(a - __half2float(hh[rr]));
      }
      memcpy(h, hh, 32);
      memcpy(l, ll, 32);
    } else {
      float hh[RPW], ll[RPW];
#pragma unroll
      for (int rr = 0; rr < RPW; ++rr) {
        hh[rr] = to_tf32(v[rr][c]);
        ll[rr] = to_tf32(v[rr][c] - hh[rr]);
      }
      memcpy(h, hh, 32);
      memcpy(l, ll, 32);
    }
    uint4* dh = reinterpret_cast<uint4*>(sm_hi + cl * kSplitColBytes + warp * 32);
    uint4* dl = reinterpret_cast<uint4*>(sm_lo + cl * kSplitColBytes + warp * 32);
    dh[0] = h[0]; dh[1] = h[1];
    dl[0] = l[0]; dl[1] = l[1];
    ysum[warp][cl] = zacc[c];
  }
  __syncthreads();
  // k-block-major output [R_pad/BK][D][BK]: for one k-block the 128 features of this block are 16 KB contiguous
  const int ncol = (D - c0 < kColBlock) ? D - c0 : kColBlock;
#pragma unroll
  for (int kb = 0; kb < 2; ++kb) {
    const size_t obase = ((size_t)(rb * 2 + kb) * D + c0) * 128;
#pragma unroll
    for (int pass = 0; pass < 4; ++pass) {
      const int piece = pass * 256 + threadIdx.x, cl = piece >> 3, part = piece & 7;
      if (cl < ncol) {
        const int so = cl * kSplitColBytes + kb * 128 + part * 16;
        *reinterpret_cast<uint4*>(At_hi + obase + (size_t)piece * 16) = *reinterpret_cast<const uint4*>(sm_hi + so);
        *reinterpret_cast<uint4*>(At_lo + obase + (size_t)piece * 16) = *reinterpret_cast<const uint4*>(sm_lo + so);
      }
    }
  }
  if (zty_part != nullptr && threadIdx.x < ncol) {
    float t = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) t += ysum[w][threadIdx.x];
    zty_part[(size_t)rb * D + c0 + threadIdx.x] = t;
  }
}

// Zty[i] (+)= sum over row blocks of the partials, in fp64, fixed order: deterministic and independent of the grid.
__global__ void __launch_bounds__(256)
zty_reduce_kernel(const float* __restrict__ part, long long n_rb, int D, float* __restrict__ Zty, int accumulate) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= D) return;
  double t = accumulate ? (double)Zty[i] : 0.0;
  for (long long rb = 0; rb < n_rb; ++rb) t += (double)part[(size_t)rb * D + i];
  Zty[i] = (float)t;
}

// ---------------------------------------------------------------------------------------------------
// 2. the tcgen05 kernel
// ---------------------------------------------------------------------------------------------------
// Tiles touching the lower triangle of C: tile (tj, ti) covers C rows [256 tj, +256) x cols [128 ti, +128);
// it is needed iff 128 ti <= 256 tj + 255, i.e. ti <= 2 tj + 1.
__host__ __device__ inline int tiles_in_row(int tj, int n_ti) { return (2 * tj + 2 < n_ti) ? 2 * tj + 2 : n_ti; }

// Tile order.  The ~148 tiles in flight should touch as few distinct operand rows of A^T as possible (they are
// re-read from L2, and from DRAM once per wave): tile rows are grouped in bands of kBandRows, and inside a band the
// tiles run column by column, so a wave covers a roughly square patch (about 8 J-blocks x 18 I-blocks) instead of
// two or three full-width rows.
constexpr int kBandRows = 8;
__host__ __device__ inline void tile_decode(int tile, int n_ti, int n_tj, int* tj_out, int* ti_out) {
  int r0 = 0, r1 = 0;
  for (r0 = 0; r0 < n_tj; r0 += kBandRows) {
    r1 = r0 + kBandRows < n_tj ? r0 + kBandRows : n_tj;
    int cnt = 0;
    for (int tj = r0; tj < r1; ++tj) cnt += tiles_in_row(tj, n_ti);
    if (tile < cnt) break;
    tile -= cnt;
  }
  for (int ti = 0; ti < n_ti; ++ti) {
    const int lo = (ti / 2 > r0) ? ti / 2 : r0;  // first tile row of the band that needs column ti
    const int cnt = r1 - lo;
    if (cnt <= 0) continue;
    if (tile < cnt) { *tj_out = lo + tile; *ti_out = ti; return; }
    tile -= cnt;
  }
  *tj_out = r1 - 1; *ti_out = 0;  // not reached for tile < n_tiles
}

// Pair tiles: (tj, tip) covers C rows [256 tj, +256) x cols [256 tip, +256), needed iff tip <= tj; same band order.
__host__ __device__ inline int ptiles_in_row(int tj, int n_tip) { return tj + 1 < n_tip ? tj + 1 : n_tip; }
__host__ __device__ inline void tile_decode2(int tile, int n_tip, int n_tj, int* tj_out, int* tip_out) {
  int r0 = 0, r1 = 0;
  for (r0 = 0; r0 < n_tj; r0 += kBandRows) {
    r1 = r0 + kBandRows < n_tj ? r0 + kBandRows : n_tj;
    int cnt = 0;
    for (int tj = r0; tj < r1; ++tj) cnt += ptiles_in_row(tj, n_tip);
    if (tile < cnt) break;
    tile -= cnt;
  }
  for (int tip = 0; tip < n_tip; ++tip) {
    const int lo = tip > r0 ? tip : r0;      // first tile row of the band that needs column pair tip
    const int cnt = r1 - lo;
    if (cnt <= 0) continue;
    if (tile < cnt) { *tj_out = lo + tile; *tip_out = tip; return; }
    tile -= cnt;
  }
  *tj_out = r1 - 1; *tip_out = 0;
}

// tile of this CTA: rows [256 tj, +256) x cols [128 ti, +128); pairs: ti = 2 tip + rank (ti >= n_ti: nothing stored)
template <bool kPair>
__device__ __forceinline__ void decode_my_tile(int tile, int n_ti, int n_tj, int rank, int* tj, int* ti) {
  if constexpr (kPair) {
    int tip;
    tile_decode2(tile, (n_ti + 1) / 2, n_tj, tj, &tip);
    *ti = 2 * tip + rank;
  } else {
    tile_decode(tile, n_ti, n_tj, tj, ti);
  }
}

template <bool F16, bool kPair>
__global__ void __launch_bounds__(kSyrkThreads, 1)
syrk_tcgen05_kernel(const __grid_constant__ CUtensorMap map_hi, const __grid_constant__ CUtensorMap map_lo,
                    float* __restrict__ C, int D, int n_kb /* BK-row blocks in the panel */, int n_tiles,
                    int first_store, const float* __restrict__ inv_scale /* [n_chunks][n_cb], F16 only */, int n_cb) {
  using M = SplitMode<F16>;
  static_assert(!kPair || F16, "CTA pairs: fp16 container only");
  constexpr int kb_per_chunk = kChunkRows / M::kBK;
  constexpr int kSt = kPair ? kStagesP : kStages;
  constexpr uint32_t kSB = kPair ? kStageBytesP : kStageBytes;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kSt * kSB);
  uint64_t* full_bar = bars;                 // [kSt]  TMA -> MMA
  uint64_t* empty_bar = bars + kSt;          // [kSt]  MMA -> TMA (pairs: multicast commit)
  uint64_t* tfull_bar = bars + 2 * kSt;      // [2]    MMA -> epilogue (pairs: multicast commit)
  uint64_t* tempty_bar = bars + 2 * kSt + 2; // [2]    epilogue -> MMA (pairs: the epilogues of both CTAs -> leader)
  uint64_t* pfull_bar = bars + 2 * kSt + 4;  // [kSt]  pairs, leader: the peer's stage has landed
  uint32_t* tmem_ptr_smem = reinterpret_cast<uint32_t*>(bars + 3 * kSt + 4);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_ti = (D + kBM - 1) / kBM, n_tj = (D + kBN - 1) / kBN;
  const int n_chunks = (n_kb + kb_per_chunk - 1) / kb_per_chunk;
  // work unit = CTA (single) or CTA pair; `rank` = position in the pair
  const int rank = kPair ? (int)cluster_ctarank() : 0;
  const int unit = kPair ? (int)(blockIdx.x >> 1) : (int)blockIdx.x;
  const int n_units = kPair ? (int)(gridDim.x >> 1) : (int)gridDim.x;
  if (threadIdx.x == 0) {
    for (int s = 0; s < kSt; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); mbar_init(&pfull_bar[s], 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(&tfull_bar[b], 1); mbar_init(&tempty_bar[b], kPair ? 16 : 8); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (warp == 2) {  // TMEM: all 512 columns = two 128 x 256 fp32 accumulators
    if constexpr (kPair) {
      asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_ptr_smem))
                   : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    } else {
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_ptr_smem))
                   : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
  }
  tcgen05_fence_before();
  __syncthreads();
  if constexpr (kPair) cluster_sync_all();   // the peer's barriers exist before anything arrives on them
  tcgen05_fence_after();
  const uint32_t tmem_base = *tmem_ptr_smem;

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      asm volatile("prefetch.tensormap [%0];" ::"l"(&map_hi) : "memory");
      asm volatile("prefetch.tensormap [%0];" ::"l"(&map_lo) : "memory");
      uint32_t kbc = 0;  // running k-block counter -> stage / phase
      for (int tile = unit; tile < n_tiles; tile += n_units) {
        int tj, rem;
        decode_my_tile<kPair>(tile, n_ti, n_tj, rank, &tj, &rem);
        const int I0 = rem * kBM, J0 = tj * kBN;
        for (int kb = 0; kb < n_kb; ++kb, ++kbc) {
          const uint32_t s = kbc % kSt, ph = (kbc / kSt) & 1;
          mbar_wait(&empty_bar[s], ph ^ 1);
          uint8_t* st = smem + s * kSB;
          mbar_expect_tx(&full_bar[s], kSB);
          // tensor = [n_kb * D][BK]: box row index = kb * D + feature.  Features past D alias the next k-block
          // (finite values; those accumulator rows / columns are masked at the store), past the end TMA fills zeros.
          const int base = kb * D;
          tma_load_2d(st, &map_hi, &full_bar[s], 0, base + I0);
          tma_load_2d(st + kTileABytes, &map_lo, &full_bar[s], 0, base + I0);
          if constexpr (kPair) {     // this CTA's half of the J operand
            tma_load_2d(st + 2 * kTileABytes, &map_hi, &full_bar[s], 0, base + J0 + 128 * rank);
            tma_load_2d(st + 3 * kTileABytes, &map_lo, &full_bar[s], 0, base + J0 + 128 * rank);
          } else {
            tma_load_2d(st + 2 * kTileABytes, &map_hi, &full_bar[s], 0, base + J0);
            tma_load_2d(st + 2 * kTileABytes + kTileABytes, &map_hi, &full_bar[s], 0, base + J0 + 128);
            tma_load_2d(st + 2 * kTileABytes + kTileBBytes, &map_lo, &full_bar[s], 0, base + J0);
            tma_load_2d(st + 2 * kTileABytes + kTileBBytes + kTileABytes, &map_lo, &full_bar[s], 0, base + J0 + 128);
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    // The whole warp runs the loop in lock-step and one elected lane issues, so that every operand of tcgen05.mma /
    // commit lives in uniform registers (under `if (lane == 0)` the compiler wraps each MMA in a vote / elect / R2UR
    // loop because it cannot prove uniformity).
    {
      const bool leader = elect_one_sync();
      const uint32_t tmem_base_u = __shfl_sync(0xffffffffu, tmem_base, 0);
      const int rank_u = __shfl_sync(0xffffffffu, rank, 0);
      // pairs: one MMA has M = 256 (the I tiles of both CTAs) and N = 256 (both halves of the J operand)
      constexpr uint32_t kIdescP = (1u << 4) | (M::kFmt << 7) | (M::kFmt << 10) | ((uint32_t)(256 >> 3) << 17) |
                                   ((uint32_t)(256 >> 4) << 24);
      uint32_t kbc = 0, item = 0;
      for (int tile = unit; tile < n_tiles; tile += n_units) {
        for (int ch = 0; ch < n_chunks; ++ch, ++item) {
          const uint32_t buf = item & 1, tph = (item >> 1) & 1;
          if (rank_u == 0) {
            mbar_wait(&tempty_bar[buf], tph ^ 1);  // the epilogue(s) have drained this accumulator
            tcgen05_fence_after();
          }
          const uint32_t tmem_d = tmem_base_u + buf * kBN;
          const int kb_end = (ch + 1) * kb_per_chunk < n_kb ? (ch + 1) * kb_per_chunk : n_kb;
          for (int kb = ch * kb_per_chunk; kb < kb_end; ++kb, ++kbc) {
            const uint32_t s = kbc % kSt, ph = (kbc / kSt) & 1;
            mbar_wait(&full_bar[s], ph);
            if constexpr (kPair) {
              if (rank_u != 0) {           // peer: my half of the stage is in my shared memory -- tell the leader
                if (leader) mbar_arrive_remote(&pfull_bar[s], 0);
                __syncwarp();
                continue;
              }
              mbar_wait(&pfull_bar[s], ph);
            }
            tcgen05_fence_after();
            const uint32_t base = smem_u32(smem + s * kSB);
            const uint64_t a_hi = make_kmajor_sw128_desc(base);
            const uint64_t a_lo = make_kmajor_sw128_desc(base + kTileABytes);
            const uint64_t b_hi = make_kmajor_sw128_desc(base + 2 * kTileABytes);
            const uint64_t b_lo = make_kmajor_sw128_desc(base + 2 * kTileABytes + (kPair ? kTileABytes : kTileBBytes));
            if (leader) {
#pragma unroll
              for (int kk = 0; kk < M::kBK / M::kUmmaK; ++kk) {
                const uint64_t adv = (uint64_t)((kk * 32) >> 4);  // +32 bytes per K step, in 16 B units
                const uint32_t acc0 = (kb > ch * kb_per_chunk || kk > 0) ? 1u : 0u;
                if constexpr (kPair) {
                  umma2<true>(tmem_d, a_lo + adv, b_hi + adv, kIdescP, acc0);   // small terms first
                  umma2<true>(tmem_d, a_hi + adv, b_lo + adv, kIdescP, 1u);
                  umma2<true>(tmem_d, a_hi + adv, b_hi + adv, kIdescP, 1u);
                } else {
                  umma<F16>(tmem_d, a_lo + adv, b_hi + adv, M::kIdesc, acc0);   // small terms first
                  umma<F16>(tmem_d, a_hi + adv, b_lo + adv, M::kIdesc, 1u);
                  umma<F16>(tmem_d, a_hi + adv, b_hi + adv, M::kIdesc, 1u);
                }
              }
              // smem stage reusable once these MMAs have read it (pairs: in both CTAs)
              if constexpr (kPair) tcgen05_commit2(&empty_bar[s]); else tcgen05_commit(&empty_bar[s]);
            }
            __syncwarp();
          }
          if (leader && rank_u == 0) {   // accumulator(s) complete
            if constexpr (kPair) tcgen05_commit2(&tfull_bar[buf]); else tcgen05_commit(&tfull_bar[buf]);
          }
          __syncwarp();
        }
      }
    }
  } else {
    // ===================== epilogue warps 2..9 =====================
    // Two warps per TMEM lane quarter; each owns half of the 256 accumulator columns.  Chunk partials are summed
    // in REGISTERS (128 fp32 per thread, round-to-nearest) so that draining TMEM every 128 rows costs only
    // tcgen05.ld + FADD (FFMA with the chunk's power-of-two scale in fp16 mode); C is touched once per tile.
    const int quarter = warp & 3;  // TMEM lanes [32 q, 32 q + 32) are the ones this warp may read
    const int chalf = (warp - 2) >> 2;  // 0: columns [0,128), 1: columns [128,256)
    const int i_loc = quarter * 32 + lane;
    uint32_t item = 0;
    for (int tile = unit; tile < n_tiles; tile += n_units) {
      int tj, rem;
      decode_my_tile<kPair>(tile, n_ti, n_tj, rank, &tj, &rem);
      const int I0 = rem * kBM, J0 = tj * kBN + chalf * 128;
      const int col = I0 + i_loc;  // column of C this thread writes (transposed store)
      const int cbI = rem, cbJ = 2 * tj + chalf;  // 128-column blocks of the two operands
      float acc[128];
#pragma unroll
      for (int j = 0; j < 128; ++j) acc[j] = 0.f;
      for (int ch = 0; ch < n_chunks; ++ch, ++item) {
        float f = 1.f;
        if constexpr (F16)
          f = (cbI < n_cb ? __ldg(inv_scale + (size_t)ch * n_cb + cbI) : 1.f) *
              (cbJ < n_cb ? __ldg(inv_scale + (size_t)ch * n_cb + cbJ) : 1.f);
        const uint32_t buf = item & 1, tph = (item >> 1) & 1;
        mbar_wait(&tfull_bar[buf], tph);
        tcgen05_fence_after();
        const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16) + buf * kBN + chalf * 128;
#pragma unroll
        for (int c0 = 0; c0 < 128; c0 += 32) {
          uint32_t r[32];
          tmem_ld_32x32b_x32(taddr + c0, r);
          tmem_ld_wait();
#pragma unroll
          for (int jj = 0; jj < 32; ++jj) {
            if constexpr (F16) acc[c0 + jj] = fmaf(__uint_as_float(r[jj]), f, acc[c0 + jj]);
            else acc[c0 + jj] += __uint_as_float(r[jj]);
          }
        }
        tcgen05_fence_before();  // all TMEM reads of this warp are done: hand the accumulator back
        __syncwarp();
        if (lane == 0) {
          if (kPair && rank != 0) mbar_arrive_remote(&tempty_bar[buf], 0); else mbar_arrive(&tempty_bar[buf]);
        }
      }
      if (col < D) {
        float* dst = C + (size_t)J0 * D + col;
        if (!first_store) {
#pragma unroll
          for (int j = 0; j < 128; ++j)
            if (J0 + j < D) acc[j] += __ldcg(dst + (size_t)j * D);
        }
#pragma unroll
        for (int j = 0; j < 128; ++j)
          if (J0 + j < D) __stcg(dst + (size_t)j * D, acc[j]);
      }
    }
  }

  tcgen05_fence_before();
  __syncthreads();
  if constexpr (kPair) cluster_sync_all();   // nobody leaves while the peer may still touch its memory
  if (warp == 2) {
    tcgen05_fence_after();
    if constexpr (kPair)
      asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
    else
      asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
  }
}

// ---------------------------------------------------------------------------------------------------
// 3. mirror: C[i, j] = C[j, i] for i < j (32 x 32 blocks through shared memory)
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
mirror_lower_kernel(float* __restrict__ C, int D) {
  __shared__ float t[32][33];
  const int bi = blockIdx.y, bj = blockIdx.x;  // destination block rows bi, cols bj; needs bj >= bi
  if (bj < bi) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int rr = warp; rr < 32; rr += 8) {  // source block: rows 32 bj + rr, cols 32 bi + lane
    const int sr = bj * 32 + rr, sc = bi * 32 + lane;
    t[rr][lane] = (sr < D && sc < D) ? C[(size_t)sr * D + sc] : 0.f;
  }
  __syncthreads();
  for (int rr = warp; rr < 32; rr += 8) {
    const int dr = bi * 32 + rr, dc = bj * 32 + lane;
    if (dr < D && dc < D && dr < dc) C[(size_t)dr * D + dc] = t[lane][rr];
  }
}

// ---------------------------------------------------------------------------------------------------
// 4. multi-GPU exchange helpers: the lower triangle of ZtZ packed row by row (row i: i + 1 entries at offset
//    i (i + 1) / 2), so that the one all-reduce of the data-parallel training step moves D (D + 1) / 2 values
//    instead of D^2; unpack writes both triangles (exactly symmetric again).
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
pack_lower_kernel(const float* __restrict__ C, int D, float* __restrict__ packed) {
  const int i = blockIdx.y;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j <= i) packed[(size_t)i * (i + 1) / 2 + j] = C[(size_t)i * D + j];
}
__global__ void __launch_bounds__(256)
unpack_lower_kernel(const float* __restrict__ packed, int D, float* __restrict__ C) {
  __shared__ float t[32][33];
  const int bi = blockIdx.y, bj = blockIdx.x;  // lower-triangle source block: rows 32 bi, cols 32 bj, bj <= bi
  if (bj > bi) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int rr = warp; rr < 32; rr += 8) {
    const int i = bi * 32 + rr, j = bj * 32 + lane;
    float v = 0.f;
    if (i < D && j <= i) {
      v = packed[(size_t)i * (i + 1) / 2 + j];
      C[(size_t)i * D + j] = v;
    }
    t[rr][lane] = v;
  }
  __syncthreads();
  for (int rr = warp; rr < 32; rr += 8) {      // mirrored block: rows 32 bj + rr, cols 32 bi + lane
    const int i = bj * 32 + rr, j = bi * 32 + lane;
    if (i < D && j < D && i < j) C[(size_t)i * D + j] = t[lane][rr];
  }
}
int syrk_pack_lower(const float* C, int32_t D, float* packed, cudaStream_t st) {
  dim3 g((unsigned)((D + 255) / 256), (unsigned)D);
  pack_lower_kernel<<<g, 256, 0, st>>>(C, D, packed);
  QMLL_LAUNCH_CHECK("pack_lower_kernel");
  return QMLL_OK;
}
int syrk_unpack_lower(const float* packed, int32_t D, float* C, cudaStream_t st) {
  dim3 g((unsigned)((D + 31) / 32), (unsigned)((D + 31) / 32));
  unpack_lower_kernel<<<g, 256, 0, st>>>(packed, D, C);
  QMLL_LAUNCH_CHECK("unpack_lower_kernel");
  return QMLL_OK;
}

// ---------------------------------------------------------------------------------------------------
// Host side
// ---------------------------------------------------------------------------------------------------
int device_sm_count();

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (fn) return fn;
  void* sym = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres);
  if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || sym == nullptr) {
    note_cuda_error(e != cudaSuccess ? e : cudaErrorUnknown, "cudaGetDriverEntryPoint(cuTensorMapEncodeTiled)");
    return nullptr;
  }
  fn = reinterpret_cast<EncodeTiledFn>(sym);
  return fn;
}

// At as [n_kb * D][BK] elements, inner (contiguous) dimension = the BK rows of a k-block (128 bytes).
// Box = BK rows x 128 features, SWIZZLE_128B.
static int make_map(CUtensorMap* map, void* base, int D, long long n_kb, bool f16) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return QMLL_ERR_CUDA;
  const cuuint32_t bk = f16 ? 64u : 32u;
  cuuint64_t dims[2] = {(cuuint64_t)bk, (cuuint64_t)D * (cuuint64_t)n_kb};
  cuuint64_t strides[1] = {128};
  cuuint32_t box[2] = {bk, 128u};
  cuuint32_t estr[2] = {1u, 1u};
  CUresult r = fn(map, f16 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, base, dims, strides,
                  box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                  CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    note_cuda_error(cudaErrorInvalidValue, "cuTensorMapEncodeTiled");
    return QMLL_ERR_CUDA;
  }
  return QMLL_OK;
}

// Optional per-launch timing of the tcgen05 kernel (bench.py's roofline): events on the caller's stream.
static std::mutex g_timing_mutex;
static bool g_timing = false;
struct TimedLaunch { cudaEvent_t a, b; };
static TimedLaunch g_timed[4096];
static int g_n_timed = 0;
void syrk_set_timing(bool on) {
  std::lock_guard<std::mutex> lock(g_timing_mutex);
  g_timing = on;
}
int syrk_collect_timing(double* total_ms, int* launches) {
  std::lock_guard<std::mutex> lock(g_timing_mutex);
  double tot = 0.0;
  for (int i = 0; i < g_n_timed; ++i) {
    float ms = 0.f;
    QMLL_CUDA_TRY(cudaEventSynchronize(g_timed[i].b));
    QMLL_CUDA_TRY(cudaEventElapsedTime(&ms, g_timed[i].a, g_timed[i].b));
    tot += ms;
    cudaEventDestroy(g_timed[i].a);
    cudaEventDestroy(g_timed[i].b);
  }
  *total_ms = tot;
  *launches = g_n_timed;
  g_n_timed = 0;
  return QMLL_OK;
}

// Workspace layout of one panel of `rp` padded rows:  At_hi | At_lo | inv_scale [rp/128][n_cb] | zty_part [n_rb][D]
struct PanelLayout {
  size_t op_bytes, scale_bytes, part_bytes;
  size_t total() const { return 2 * op_bytes + scale_bytes + part_bytes + 4 * 256; }
};
static long long tile_rows(int mode) { return mode != QMLL_NE_SPLIT_TF32 ? 128 : 64; }
static long long pad_rows(long long r, int mode) { return (r + tile_rows(mode) - 1) / tile_rows(mode) * tile_rows(mode); }
static PanelLayout panel_layout(long long rp, int D, int mode) {
  const int eb = mode != QMLL_NE_SPLIT_TF32 ? 2 : 4;
  const int n_cb = (D + kColBlock - 1) / kColBlock;
  PanelLayout l;
  l.op_bytes = align_up((size_t)D * rp * eb, 256);
  l.scale_bytes = align_up((size_t)((rp + kChunkRows - 1) / kChunkRows) * n_cb * sizeof(float), 256);
  l.part_bytes = align_up((size_t)(rp / tile_rows(mode)) * D * sizeof(float), 256);
  return l;
}

size_t syrk_min_workspace(int32_t D, int mode) { return panel_layout(kPanelRows, D, mode).total(); }
size_t syrk_full_workspace(int64_t rows, int32_t D, int mode) {
  long long rp = pad_rows(rows < 1 ? 1 : rows, mode);
  if (rp < kPanelRows) rp = kPanelRows;
  return panel_layout(rp, D, mode).total();
}

template <bool F16, bool kPair>
static int syrk_impl(const float* A, const float* y, int64_t rows, int32_t D, int accumulate, float* ZtZ, float* Zty,
                     void* ws, size_t ws_bytes, cudaStream_t st) {
  using M = SplitMode<F16>;
  constexpr int mode = F16 ? QMLL_NE_SPLIT_F16 : QMLL_NE_SPLIT_TF32;
  // rows per panel: as many as the workspace holds, a multiple of kPanelRows unless everything fits -- but never more
  // than kMaxPanelRows: the CTAs of the persistent kernel drift apart along the rows, and once the operand rows they
  // are reading no longer fit L2 together every CTA streams from DRAM on its own (config 3, 100 000 rows: 0.76 of the
  // tensor peak in one panel).  Panels re-synchronise them; ZtZ is read-modify-written once per extra panel.
  long long panel = pad_rows(rows, mode);
  if (panel > kMaxPanelRows) {
    const long long n_pan = (panel + kMaxPanelRows - 1) / kMaxPanelRows;
    panel = ((panel + n_pan - 1) / n_pan + kPanelRows - 1) / kPanelRows * kPanelRows;
  }
  if (panel_layout(panel, D, mode).total() > ws_bytes) {
    const size_t per_row = (size_t)2 * D * M::kElemBytes;   // lower bound of the bytes one more row costs
    panel = (long long)(ws_bytes / per_row) / kPanelRows * kPanelRows + kPanelRows;
    while (panel >= kPanelRows && panel_layout(panel, D, mode).total() > ws_bytes) panel -= kPanelRows;
    if (panel < kPanelRows) return QMLL_ERR_WORKSPACE;
  }
  // the split pass puts row blocks on grid.x (2^31-1 blocks), feature blocks on grid.y (D <= 65535 * 128)
  const int n_cb = (D + kColBlock - 1) / kColBlock;
  if (n_cb > 65535) return QMLL_ERR_UNSUPPORTED;
  const PanelLayout lay = panel_layout(panel, D, mode);
  Carver carve(ws, ws_bytes);
  uint8_t* At_hi = carve.take<uint8_t>(lay.op_bytes);
  uint8_t* At_lo = carve.take<uint8_t>(lay.op_bytes);
  float* inv_scale = carve.take<float>(lay.scale_bytes / sizeof(float));
  float* zty_part = carve.take<float>(lay.part_bytes / sizeof(float));
  if (!carve.fits()) return QMLL_ERR_WORKSPACE;

  const int n_ti = (D + kBM - 1) / kBM, n_tj = (D + kBN - 1) / kBN;
  int n_tiles = 0;
  for (int tj = 0; tj < n_tj; ++tj) n_tiles += kPair ? ptiles_in_row(tj, (n_ti + 1) / 2) : tiles_in_row(tj, n_ti);
  const int max_units = kPair ? device_sm_count() / 2 : device_sm_count();
  const int grid = (n_tiles < max_units ? n_tiles : max_units) * (kPair ? 2 : 1);
  constexpr uint32_t smem_bytes = kPair ? kSmemBytesP : kSmemBytes;
  auto kern = syrk_tcgen05_kernel<F16, kPair>;
  QMLL_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes));
  QMLL_CUDA_TRY(cudaFuncSetAttribute(split_kernel<F16>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSplitSmem));
  int first_store = accumulate ? 0 : 1;
  int zty_acc = accumulate ? 1 : 0;
  for (int64_t r0 = 0; r0 < rows; r0 += panel) {
    const long long pr = (rows - r0 < panel) ? rows - r0 : panel;
    const long long rp = pad_rows(pr, mode);
    const long long n_rb = rp / M::kTileRows;
    dim3 g1((unsigned)n_rb, (unsigned)n_cb);
    split_kernel<F16><<<g1, 256, kSplitSmem, st>>>(A + (size_t)r0 * D, y ? y + r0 : nullptr, pr, D, At_hi, At_lo,
                                                  inv_scale, n_cb, (y && Zty) ? zty_part : nullptr);
    QMLL_LAUNCH_CHECK("split_kernel");
    if (y && Zty) {
      zty_reduce_kernel<<<(D + 255) / 256, 256, 0, st>>>(zty_part, n_rb, D, Zty, zty_acc);
      QMLL_LAUNCH_CHECK("zty_reduce_kernel");
      zty_acc = 1;
    }
    CUtensorMap map_hi, map_lo;
    const long long n_kb = rp / M::kBK;
    int rc = make_map(&map_hi, At_hi, D, n_kb, F16);
    if (rc != QMLL_OK) return rc;
    rc = make_map(&map_lo, At_lo, D, n_kb, F16);
    if (rc != QMLL_OK) return rc;
    bool timed = false;
    {
      std::lock_guard<std::mutex> lock(g_timing_mutex);
      timed = g_timing && g_n_timed < 4096;
      if (timed) {
        QMLL_CUDA_TRY(cudaEventCreate(&g_timed[g_n_timed].a));
        QMLL_CUDA_TRY(cudaEventCreate(&g_timed[g_n_timed].b));
        QMLL_CUDA_TRY(cudaEventRecord(g_timed[g_n_timed].a, st));
      }
    }
    {
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((unsigned)grid);
      cfg.blockDim = dim3(kSyrkThreads);
      cfg.dynamicSmemBytes = smem_bytes;
      cfg.stream = st;
      cudaLaunchAttribute attr[1];
      attr[0].id = cudaLaunchAttributeClusterDimension;
      attr[0].val.clusterDim.x = kPair ? 2 : 1;
      attr[0].val.clusterDim.y = 1;
      attr[0].val.clusterDim.z = 1;
      cfg.attrs = attr;
      cfg.numAttrs = 1;
      const int n_kb_i = (int)n_kb;
      const float* inv_c = inv_scale;
      QMLL_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, map_hi, map_lo, ZtZ, (int)D, n_kb_i, n_tiles, first_store, inv_c, n_cb));
    }
    QMLL_LAUNCH_CHECK("syrk_tcgen05_kernel");
    if (timed) {
      std::lock_guard<std::mutex> lock(g_timing_mutex);
      QMLL_CUDA_TRY(cudaEventRecord(g_timed[g_n_timed].b, st));
      ++g_n_timed;
    }
    first_store = 0;
  }
  dim3 g3((unsigned)((D + 31) / 32), (unsigned)((D + 31) / 32));
  mirror_lower_kernel<<<g3, 256, 0, st>>>(ZtZ, D);
  QMLL_LAUNCH_CHECK("mirror_lower_kernel");
  return QMLL_OK;
}

int syrk_normal_equations(const float* A, const float* y, int64_t rows, int32_t D, int accumulate, float* ZtZ,
                          float* Zty, void* ws, size_t ws_bytes, int mode, cudaStream_t st) {
  if (!accumulate) {
    if (Zty) QMLL_CUDA_TRY(cudaMemsetAsync(Zty, 0, (size_t)D * sizeof(float), st));
    if (rows == 0) QMLL_CUDA_TRY(cudaMemsetAsync(ZtZ, 0, (size_t)D * D * sizeof(float), st));
  }
  if (rows == 0) return QMLL_OK;
  if (ws == nullptr || ((uintptr_t)ws & 255) != 0) return QMLL_ERR_WORKSPACE;
  if (mode == QMLL_NE_SPLIT_F16) return syrk_impl<true, false>(A, y, rows, D, accumulate, ZtZ, Zty, ws, ws_bytes, st);
  if (mode == QMLL_NE_SPLIT_F16_PAIRS) return syrk_impl<true, true>(A, y, rows, D, accumulate, ZtZ, Zty, ws, ws_bytes, st);
  return syrk_impl<false, false>(A, y, rows, D, accumulate, ZtZ, Zty, ws, ws_bytes, st);
}

}  // namespace qmll
