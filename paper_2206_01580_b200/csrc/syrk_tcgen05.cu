// syrk_tcgen05.cu -- step a8: the normal equations ZtZ (+)= A^T A, Zty (+)= A^T y (eq. 16,
// eq. 17) on the 5th-generation tensor cores in 3xTF32 (fp32-level accuracy; the paper's FP32
// round-off remark L351 is answered by splitting every operand into TF32 hi + lo parts and by cutting the
// row dimension into chunks whose partial products are summed in fp32 round-to-nearest).
//
// Pipeline of one call (per panel of rows that fits the workspace):
//   1. split_transpose_kernel: A[rows, D] -> At_hi, At_lo [R_pad/32][D][32] (K-major for the MMA: the contraction
//      index `row` is the contiguous one inside each 32-row block; one TMA box is 16 KB contiguous), hi = tf32(a), lo = tf32(a - hi); Zty += A^T y rides along.
//   2. syrk_tcgen05_kernel: persistent, warp-specialised.  One CTA owns a 128 x 256 tile T = At[I,:] At[J,:]^T
//      for ALL rows: TMA (SWIZZLE_128B) -> 2-stage smem ring -> tcgen05.mma kind::tf32 (hi*hi + hi*lo +
//      lo*hi) into one of two 256-column TMEM accumulators; every 1024 rows the accumulator is drained by
//      4 epilogue warps (tcgen05.ld) and added into C in fp32 while the next chunk is already running.
//      The tile is written transposed (C[J0+j, I0+i], coalesced along i); only tiles touching the lower
//      triangle are computed.
//   3. mirror_lower_kernel: C[i, j] = C[j, i] for i < j  -> full, exactly symmetric matrix.
#include <cuda.h>
#include <stdlib.h>

#include "qmll_common.cuh"
#include "ptx_utils.cuh"

namespace qmll {

constexpr int kBM = 128;          // tile extent along I (MMA M, TMEM lanes)
constexpr int kBN = 256;          // tile extent along J (MMA N, TMEM columns)
constexpr int kBK = 32;           // rows per pipeline stage = one 128-byte swizzle span of fp32
constexpr int kUmmaK = 8;         // rows per tcgen05.mma kind::tf32 (32 bytes)
constexpr int kStages = 2;
constexpr int kChunkRows = 1024;  // panel granularity (rows); the TMEM drain interval is chunk_rows() <= this
// Rows accumulated in TMEM before a drain.  The tensor core truncates (rounds toward zero) every accumulate, a
// bias of ~2e-8 per MMA relative to the running sum, so long same-sign sums (Gram diagonals, coherent Z columns)
// need short chunks; chunk partials are summed in fp32 round-to-nearest.  QMLL_CHUNK_ROWS overrides (tuning).
static int chunk_rows() {
  static int v = 0;
  if (v == 0) {
    v = 128;
    const char* e = getenv("QMLL_CHUNK_ROWS");
    if (e) { int t = atoi(e); if (t >= 32 && t <= 1024 && t % 32 == 0) v = t; }
  }
  return v;
}
constexpr int kRowPad = 64;       // panels are padded with zero rows to a multiple of this
constexpr int kSyrkThreads = 320; // warp 0 TMA producer, warp 1 MMA issuer, warps 2..9 epilogue
constexpr uint32_t kTileABytes = kBM * kBK * 4;             // 16 KB
constexpr uint32_t kTileBBytes = kBN * kBK * 4;             // 32 KB
constexpr uint32_t kStageBytes = 2 * kTileABytes + 2 * kTileBBytes;  // hi + lo of both operands: 96 KB
constexpr uint32_t kSmemBytes = kStages * kStageBytes + 256 + 1024;  // + barriers + alignment slack

// ---------------------------------------------------------------------------------------------------
// PTX wrappers
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
      : "memory");
}
__device__ __forceinline__ void tcgen05_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tcgen05_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tcgen05_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
               : "memory");
}
// D[tmem] (+)= A[smem desc] * B[smem desc]^T, kind::tf32, fp32 accumulate
__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                          uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(tmem_d),
      "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tmem_ld_32x32b_x32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
        "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
        "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// Shared-memory matrix descriptor, K-major, SWIZZLE_128B: rows of 128 bytes, 8-row groups 1024 bytes apart.
__device__ __forceinline__ uint64_t make_kmajor_sw128_desc(uint32_t smem_addr) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr & 0x3FFFF) >> 4);   // start address, bits [0,14)
  d |= (uint64_t)1 << 16;                        // leading byte offset (unused for swizzled K-major), bits [16,30)
  d |= (uint64_t)(1024 >> 4) << 32;              // stride byte offset = 1024 B, bits [32,46)
  d |= (uint64_t)1 << 46;                        // descriptor version (sm_100), bits [46,48)
  d |= (uint64_t)2 << 61;                        // layout type SWIZZLE_128B, bits [61,64)
  return d;
}
// Instruction descriptor: D fp32, A/B tf32, both K-major, N = 256, M = 128.
constexpr uint32_t kIdesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(kBN >> 3) << 17) |
                            ((uint32_t)(kBM >> 4) << 24);

__device__ __forceinline__ float to_tf32(float a) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(a));
  return __uint_as_float(r);
}

// ---------------------------------------------------------------------------------------------------
// 1. split + transpose (+ A^T y).  Block: 32 features x 64 rows.
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
split_transpose_kernel(const float* __restrict__ A, const float* __restrict__ y, long long rows, int D,
                       long long R_pad, float* __restrict__ At_hi, float* __restrict__ At_lo,
                       float* __restrict__ Zty) {
  __shared__ float thi[64][33], tlo[64][33];
  __shared__ float ysum[8][32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int i0 = blockIdx.x * 32;
  const long long r0 = (long long)blockIdx.y * 64;
  const int i = i0 + lane;
  float zacc = 0.f;
#pragma unroll
  for (int rr = warp; rr < 64; rr += 8) {
    const long long r = r0 + rr;
    float a = 0.f;
    if (r < rows && i < D) a = __ldcs(A + (size_t)r * D + i);
    const float hi = to_tf32(a);
    const float lo = to_tf32(a - hi);
    thi[rr][lane] = hi;
    tlo[rr][lane] = lo;
    if (y != nullptr && r < rows) zacc = fmaf(a, __ldg(y + r), zacc);
  }
  ysum[warp][lane] = zacc;
  __syncthreads();
#pragma unroll
  for (int cc = 0; cc < 4; ++cc) {
    const int c = warp * 4 + cc;
    if (i0 + c < D) {
      // k-block-major layout [R_pad/32][D][32]: the 128 features x 32 rows of one TMA box are 16 KB contiguous
      const size_t o0 = ((size_t)(r0 / 32) * D + (i0 + c)) * 32, o1 = o0 + (size_t)D * 32;
      At_hi[o0 + lane] = thi[lane][c];
      At_hi[o1 + lane] = thi[lane + 32][c];
      At_lo[o0 + lane] = tlo[lane][c];
      At_lo[o1 + lane] = tlo[lane + 32][c];
    }
  }
  if (Zty != nullptr && y != nullptr && warp == 0 && i < D) {
    float s = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) s += ysum[w][lane];
    atomicAdd(Zty + i, s);
  }
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

__global__ void __launch_bounds__(kSyrkThreads, 1)
syrk_tcgen05_kernel(const __grid_constant__ CUtensorMap map_hi, const __grid_constant__ CUtensorMap map_lo,
                    float* __restrict__ C, int D, int n_kb /* 32-row blocks in the panel */, int n_tiles,
                    int first_store, int kb_per_chunk) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kStages * kStageBytes);
  uint64_t* full_bar = bars;                 // [kStages]  TMA -> MMA
  uint64_t* empty_bar = bars + kStages;      // [kStages]  MMA -> TMA
  uint64_t* tfull_bar = bars + 2 * kStages;  // [2]        MMA -> epilogue
  uint64_t* tempty_bar = bars + 2 * kStages + 2;  // [2]   epilogue -> MMA
  uint32_t* tmem_ptr_smem = reinterpret_cast<uint32_t*>(bars + 2 * kStages + 4);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_ti = (D + kBM - 1) / kBM, n_tj = (D + kBN - 1) / kBN;
  const int n_chunks = (n_kb + kb_per_chunk - 1) / kb_per_chunk;

  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(&tfull_bar[b], 1); mbar_init(&tempty_bar[b], 8); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (warp == 2) {  // TMEM: all 512 columns = two 128 x 256 fp32 accumulators
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_ptr_smem))
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  const uint32_t tmem_base = *tmem_ptr_smem;

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      asm volatile("prefetch.tensormap [%0];" ::"l"(&map_hi) : "memory");
      asm volatile("prefetch.tensormap [%0];" ::"l"(&map_lo) : "memory");
      uint32_t kbc = 0;  // running k-block counter -> stage / phase
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        int tj, rem;
        tile_decode(tile, n_ti, n_tj, &tj, &rem);
        const int I0 = rem * kBM, J0 = tj * kBN;
        for (int kb = 0; kb < n_kb; ++kb, ++kbc) {
          const uint32_t s = kbc % kStages, ph = (kbc / kStages) & 1;
          mbar_wait(&empty_bar[s], ph ^ 1);
          uint8_t* st = smem + s * kStageBytes;
          mbar_expect_tx(&full_bar[s], kStageBytes);
          // tensor = [n_kb * D][32]: box row index = kb * D + feature.  Features past D alias the next k-block
          // (finite values; those accumulator rows / columns are masked at the store), past the end TMA fills zeros.
          const int base = kb * D;
          tma_load_2d(st, &map_hi, &full_bar[s], 0, base + I0);
          tma_load_2d(st + kTileABytes, &map_lo, &full_bar[s], 0, base + I0);
          tma_load_2d(st + 2 * kTileABytes, &map_hi, &full_bar[s], 0, base + J0);
          tma_load_2d(st + 2 * kTileABytes + kTileABytes, &map_hi, &full_bar[s], 0, base + J0 + 128);
          tma_load_2d(st + 2 * kTileABytes + kTileBBytes, &map_lo, &full_bar[s], 0, base + J0);
          tma_load_2d(st + 2 * kTileABytes + kTileBBytes + kTileABytes, &map_lo, &full_bar[s], 0, base + J0 + 128);
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (one thread) =====================
    if (lane == 0) {
      uint32_t kbc = 0, item = 0;
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        for (int ch = 0; ch < n_chunks; ++ch, ++item) {
          const uint32_t buf = item & 1, tph = (item >> 1) & 1;
          mbar_wait(&tempty_bar[buf], tph ^ 1);  // epilogue has drained this accumulator
          tcgen05_fence_after();
          const uint32_t tmem_d = tmem_base + buf * kBN;
          const int kb_end = (ch + 1) * kb_per_chunk < n_kb ? (ch + 1) * kb_per_chunk : n_kb;
          for (int kb = ch * kb_per_chunk; kb < kb_end; ++kb, ++kbc) {
            const uint32_t s = kbc % kStages, ph = (kbc / kStages) & 1;
            mbar_wait(&full_bar[s], ph);
            tcgen05_fence_after();
            const uint32_t base = smem_u32(smem + s * kStageBytes);
            const uint64_t a_hi = make_kmajor_sw128_desc(base);
            const uint64_t a_lo = make_kmajor_sw128_desc(base + kTileABytes);
            const uint64_t b_hi = make_kmajor_sw128_desc(base + 2 * kTileABytes);
            const uint64_t b_lo = make_kmajor_sw128_desc(base + 2 * kTileABytes + kTileBBytes);
#pragma unroll
            for (int kk = 0; kk < kBK / kUmmaK; ++kk) {
              const uint64_t adv = (uint64_t)((kk * kUmmaK * 4) >> 4);  // +32 bytes per K step, in 16 B units
              const uint32_t acc0 = (kb > ch * kb_per_chunk || kk > 0) ? 1u : 0u;
              umma_tf32(tmem_d, a_lo + adv, b_hi + adv, kIdesc, acc0);   // small terms first
              umma_tf32(tmem_d, a_hi + adv, b_lo + adv, kIdesc, 1u);
              umma_tf32(tmem_d, a_hi + adv, b_hi + adv, kIdesc, 1u);
            }
            tcgen05_commit(&empty_bar[s]);  // smem stage reusable once these MMAs have read it
          }
          tcgen05_commit(&tfull_bar[buf]);  // accumulator complete
        }
      }
    }
  } else {
    // ===================== epilogue warps 2..9 =====================
    // Two warps per TMEM lane quarter; each owns half of the 256 accumulator columns.  Chunk partials are summed
    // in REGISTERS (128 fp32 per thread, round-to-nearest) so that draining TMEM every few hundred rows costs only
    // tcgen05.ld + FADD; C is touched once per tile.
    const int quarter = warp & 3;  // TMEM lanes [32 q, 32 q + 32) are the ones this warp may read
    const int chalf = (warp - 2) >> 2;  // 0: columns [0,128), 1: columns [128,256)
    const int i_loc = quarter * 32 + lane;
    uint32_t item = 0;
    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
      int tj, rem;
      tile_decode(tile, n_ti, n_tj, &tj, &rem);
      const int I0 = rem * kBM, J0 = tj * kBN + chalf * 128;
      const int col = I0 + i_loc;  // column of C this thread writes (transposed store)
      float acc[128];
#pragma unroll
      for (int j = 0; j < 128; ++j) acc[j] = 0.f;
      for (int ch = 0; ch < n_chunks; ++ch, ++item) {
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
          for (int jj = 0; jj < 32; ++jj) acc[c0 + jj] += __uint_as_float(r[jj]);
        }
        tcgen05_fence_before();  // all TMEM reads of this warp are done: hand the accumulator back
        __syncwarp();
        if (lane == 0) mbar_arrive(&tempty_bar[buf]);
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
  if (warp == 2) {
    tcgen05_fence_after();
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

// At [D, R_pad] fp32, inner (contiguous) dimension = rows.  Box = 32 rows x 128 features, SWIZZLE_128B.
static int make_map(CUtensorMap* map, float* base, int D, long long R_pad) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return QMLL_ERR_CUDA;
  cuuint64_t dims[2] = {(cuuint64_t)kBK, (cuuint64_t)D * (cuuint64_t)(R_pad / kBK)};
  cuuint64_t strides[1] = {(cuuint64_t)kBK * sizeof(float)};
  cuuint32_t box[2] = {(cuuint32_t)kBK, 128u};
  cuuint32_t estr[2] = {1u, 1u};
  CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, base, dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    note_cuda_error(cudaErrorInvalidValue, "cuTensorMapEncodeTiled");
    return QMLL_ERR_CUDA;
  }
  return QMLL_OK;
}

// Optional per-launch timing of the tcgen05 kernel (bench.py's roofline): events on the caller's stream.
static bool g_timing = false;
struct TimedLaunch { cudaEvent_t a, b; };
static TimedLaunch g_timed[4096];
static int g_n_timed = 0;
void syrk_set_timing(bool on) { g_timing = on; }
int syrk_collect_timing(double* total_ms, int* launches) {
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

static long long pad_rows(long long r) { return (r + kRowPad - 1) / kRowPad * kRowPad; }

size_t syrk_min_workspace(int32_t D) { return (size_t)2 * D * kChunkRows * sizeof(float) + 1024; }
size_t syrk_full_workspace(int64_t rows, int32_t D) {
  long long rp = pad_rows(rows < 1 ? 1 : rows);
  if (rp < kChunkRows) rp = kChunkRows;
  return (size_t)2 * D * rp * sizeof(float) + 1024;
}

int syrk_normal_equations(const float* A, const float* y, int64_t rows, int32_t D, int accumulate, float* ZtZ,
                          float* Zty, void* ws, size_t ws_bytes, cudaStream_t st) {
  if (!accumulate) {
    if (Zty) QMLL_CUDA_TRY(cudaMemsetAsync(Zty, 0, (size_t)D * sizeof(float), st));
    if (rows == 0) QMLL_CUDA_TRY(cudaMemsetAsync(ZtZ, 0, (size_t)D * D * sizeof(float), st));
  }
  if (rows == 0) return QMLL_OK;
  if (ws == nullptr || ((uintptr_t)ws & 255) != 0) return QMLL_ERR_WORKSPACE;
  // rows per panel: as many as the workspace holds (two [D, R_pad] fp32 arrays), a multiple of the chunk
  long long cap = (long long)((ws_bytes > 1024 ? ws_bytes - 1024 : 0) / ((size_t)2 * D * sizeof(float)));
  long long panel = pad_rows(rows);
  if (cap < panel) {
    panel = cap / kChunkRows * kChunkRows;
    if (panel < kChunkRows) return QMLL_ERR_WORKSPACE;
  }
  float* At_hi = static_cast<float*>(ws);
  float* At_lo = At_hi + (size_t)D * panel;

  const int n_ti = (D + kBM - 1) / kBM, n_tj = (D + kBN - 1) / kBN;
  int n_tiles = 0;
  for (int tj = 0; tj < n_tj; ++tj) n_tiles += tiles_in_row(tj, n_ti);
  const int grid = n_tiles < device_sm_count() ? n_tiles : device_sm_count();
  QMLL_CUDA_TRY(cudaFuncSetAttribute(syrk_tcgen05_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)kSmemBytes));
  int first_store = accumulate ? 0 : 1;
  for (int64_t r0 = 0; r0 < rows; r0 += panel) {
    const long long pr = (rows - r0 < panel) ? rows - r0 : panel;
    const long long rp = pad_rows(pr);
    dim3 g1((unsigned)((D + 31) / 32), (unsigned)(rp / 64));
    split_transpose_kernel<<<g1, 256, 0, st>>>(A + (size_t)r0 * D, y ? y + r0 : nullptr, pr, D, rp, At_hi, At_lo,
                                              Zty);
    QMLL_LAUNCH_CHECK("split_transpose_kernel");
    CUtensorMap map_hi, map_lo;
    int rc = make_map(&map_hi, At_hi, D, rp);
    if (rc != QMLL_OK) return rc;
    rc = make_map(&map_lo, At_lo, D, rp);
    if (rc != QMLL_OK) return rc;
    const bool timed = g_timing && g_n_timed < 4096;
    if (timed) {
      QMLL_CUDA_TRY(cudaEventCreate(&g_timed[g_n_timed].a));
      QMLL_CUDA_TRY(cudaEventCreate(&g_timed[g_n_timed].b));
      QMLL_CUDA_TRY(cudaEventRecord(g_timed[g_n_timed].a, st));
    }
    syrk_tcgen05_kernel<<<grid, kSyrkThreads, kSmemBytes, st>>>(map_hi, map_lo, ZtZ, D, (int)(rp / kBK), n_tiles,
                                                              first_store, chunk_rows() / kBK);
    QMLL_LAUNCH_CHECK("syrk_tcgen05_kernel");
    if (timed) {
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

}  // namespace qmll
