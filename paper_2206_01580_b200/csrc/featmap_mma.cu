// featmap_mma.cu -- NEXT row f4 of SURVEY.md section 8(f) (variants): the random-feature map on the tensor cores,
//   Z[M, l] = sum_{I in M} sqrt(2/D) cos( (W_{e_I} x_I)[l] + b[e_I, l] )              (eq. 14, eq. 15)
// for (a) SORF: W_{e,s} = c H S_T ... H S_1 expanded once into its d x d integer matrix (exact in fp16 for d <= 256, see
// sorf_mma.cu) -- the tensor-core alternative to the ALU-bound register FWHT (the survey's "Kronecker tensor-core
// Hadamard" variant, taken to its end: the whole chain of a stack is ONE matrix); and (b) RFF: a dense Gaussian W given
// by the caller (eq. 12-14, 18 L99-121, L150-152; the paper's Fig. 1 comparison), split into fp16 hi + lo.
//
// Why it pays on B200: per feature the FWHT chain costs T log2(d) adds + T sign flips on the fp32 pipe (~1 ps at the
// measured 25 T adds/s); the explicit product costs 2 d MACs per pass on tcgen05, 2 passes for SORF (x split hi/lo, W
// exact) = 0.37 ps at d = 128.  Measured (config 3, profiles/r2_fchl19_featmap.md): 20 ms against 30.5 ms.  The epilogue
// warps are latency-bound (0.52 instructions per cycle and scheduler with the 16 epilogue warps of one CTA), so at
// d = 128 TWO CTAs share an SM (64 KB of W, 2 stages, 256 TMEM columns each: 22.8 -> 20 ms, issue rate 0.77).
//
// Dataflow: W tiles are the stationary operand (d = 128: 64 KB = 2 stacks per CTA, two CTAs per SM; d = 256: 128 KB =
// 1 stack, one CTA per SM), so
// the atoms are first SORTED BY ELEMENT inside groups of 8192 atoms (stable, so the atoms of a molecule that share an
// element stay adjacent; group-local, so that the reductions into a molecule's row of Z stay in L2) into tiles of kNT
// columns that never mix elements; x rows are gathered, scaled by one power of two per tile and split into
// fp16 hi + lo in the swizzled K-major layout (one contiguous bulk copy per k-block).  Task = (chunk of atom tiles,
// group of feature tiles): producer warp (bulk copies) / MMA warp (one elected lane issues) / 16 epilogue warps.  Epilogue
// thread = output feature: cos(c u + b) of every atom column, summed in a register over the run of columns that belong
// to the same molecule, one fp32 reduction (RED.ADD) into Z per (run, feature).  Z is zeroed first.
#include <cuda_fp16.h>

#include "qmll_common.cuh"
#include "sorf_device.cuh"
#include "tcgen05_utils.cuh"

namespace qmll {

int device_sm_count();   // sorf_dispatch.cu

constexpr int kFmMaxElem = 16;
constexpr int kFmSortThreads = 1024;
constexpr int kFmGrpBlks = 8;          // 1024-atom blocks per sort group (8192 atoms: their Z rows stay in L2)
constexpr int kFmChunkTiles = 16;      // atom tiles per task: the W tiles are loaded once per (task, element run)

__host__ __device__ constexpr int fm_nt(int d) { return d <= 128 ? 64 : 96; }   // atoms per tile (MMA N)

// ---------------------------------------------------------------------------------------------------
// 1. Sort by (atom group, element).  blk_cnt / blk_off [n_blk][E]; key_tile0[n_keys + 1] first tile of every key.
// ---------------------------------------------------------------------------------------------------
static __global__ void __launch_bounds__(kFmSortThreads)
fm_block_count_kernel(const int32_t* __restrict__ elem, long long n_atoms, int E, int* __restrict__ blk_cnt) {
  __shared__ int cnt[kFmMaxElem];
  if (threadIdx.x < kFmMaxElem) cnt[threadIdx.x] = 0;
  __syncthreads();
  const long long a = (long long)blockIdx.x * kFmSortThreads + threadIdx.x;
  if (a < n_atoms) {
    int e = __ldg(elem + a);
    e = e < 0 ? 0 : (e >= E ? E - 1 : e);
    atomicAdd(&cnt[e], 1);
  }
  __syncthreads();
  if (threadIdx.x < E) blk_cnt[(size_t)blockIdx.x * E + threadIdx.x] = cnt[threadIdx.x];
}

// Sort key = (group of kFmGrpBlks consecutive 1024-atom blocks, element): atoms are sorted by element only INSIDE a
// group (8192 atoms), so that all the reductions into the Z rows of a group's molecules happen close in time and stay in
// L2 (a global sort by element turned every reduction into a DRAM read-modify-write: 45 GB of traffic on config 3).
static __global__ void fm_group_scan_kernel(const int* __restrict__ blk_cnt, int n_blk, int n_grp, int E,
                                            int* __restrict__ blk_off, int* __restrict__ key_cnt) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;       // key = g * E + e
  if (k >= n_grp * E) return;
  const int g = k / E, e = k % E;
  int run = 0;
  for (int b = g * kFmGrpBlks; b < (g + 1) * kFmGrpBlks && b < n_blk; ++b) {
    const int t = blk_cnt[(size_t)b * E + e];
    blk_off[(size_t)b * E + e] = run;
    run += t;
  }
  key_cnt[k] = run;
}

// key_tile0[n_keys + 1]: first tile of every key (one warp, chunks of 32 keys, shuffle scan)
static __global__ void __launch_bounds__(32)
fm_tile_scan_kernel(const int* __restrict__ key_cnt, int n_keys, int nt, int* __restrict__ key_tile0) {
  const int lane = threadIdx.x;
  int carry = 0;
  for (int base = 0; base < n_keys; base += 32) {
    const int k = base + lane;
    const int tiles = k < n_keys ? (key_cnt[k] + nt - 1) / nt : 0;
    int incl = tiles;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, incl, off);
      if (lane >= off) incl += t;
    }
    if (k < n_keys) key_tile0[k] = carry + incl - tiles;
    carry += __shfl_sync(0xffffffffu, incl, 31);
  }
  if (lane == 0) key_tile0[n_keys] = carry;
}

// col_atom / col_mol [tiles * nt] (pre-set to -1)
static __global__ void __launch_bounds__(kFmSortThreads)
fm_place_kernel(const int32_t* __restrict__ elem, const int32_t* __restrict__ mol_off, long long n_atoms, int n_mol,
                int E, int nt, const int* __restrict__ blk_off, const int* __restrict__ key_tile0,
                int* __restrict__ col_atom, int* __restrict__ col_mol) {
  __shared__ int wcnt[kFmSortThreads / 32][kFmMaxElem];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int t = threadIdx.x; t < (kFmSortThreads / 32) * kFmMaxElem; t += kFmSortThreads) (&wcnt[0][0])[t] = 0;
  __syncthreads();
  const long long a = (long long)blockIdx.x * kFmSortThreads + threadIdx.x;
  int e = -1;
  if (a < n_atoms) {
    e = __ldg(elem + a);
    e = e < 0 ? 0 : (e >= E ? E - 1 : e);
  }
  const unsigned peers = __match_any_sync(0xffffffffu, e);
  const int rank = __popc(peers & ((1u << lane) - 1u));
  if (e >= 0 && rank == 0) wcnt[warp][e] = __popc(peers);
  __syncthreads();
  if (threadIdx.x < E) {
    int run = 0;
    for (int w = 0; w < kFmSortThreads / 32; ++w) { const int t = wcnt[w][threadIdx.x]; wcnt[w][threadIdx.x] = run; run += t; }
  }
  __syncthreads();
  if (e >= 0) {
    const int key = (blockIdx.x / kFmGrpBlks) * E + e;
    const size_t pos = (size_t)__ldg(key_tile0 + key) * nt + __ldg(blk_off + (size_t)blockIdx.x * E + e) + wcnt[warp][e] + rank;
    col_atom[pos] = (int)a;
    col_mol[pos] = owner_molecule(mol_off, n_mol, (int)a);
  }
}

// tile_elem [tiles_max]: element of the key that owns the tile (-1 beyond the last tile)
static __global__ void fm_tile_elem_kernel(const int* __restrict__ key_tile0, int n_keys, int E, int tiles_max,
                                           int* __restrict__ tile_elem) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= tiles_max) return;
  int e = -1;
  if (t < __ldg(key_tile0 + n_keys)) {
    int lo = 0, hi = n_keys;                 // smallest k in [0, n_keys] with key_tile0[k] > t
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if (__ldg(key_tile0 + mid) > t) hi = mid; else lo = mid + 1;
    }
    e = (lo - 1) % E;
  }
  tile_elem[t] = e;
}

// Runs of columns that belong to the same molecule, per tile: end_mask[tile][4] has bit c set if column c is the last
// column of its run (the tile's last column always is); run_mol[tile * nt + k] = molecule of the k-th run (-1: padding).
// The epilogue then needs no per-column comparison: one bit test per column, one load per run.
static __global__ void __launch_bounds__(128)
fm_runs_kernel(const int* __restrict__ col_mol, const int* __restrict__ n_tiles_ptr, int nt, int mult,
               uint32_t* __restrict__ end_mask, int* __restrict__ run_mol) {
  const int lane = threadIdx.x & 31;
  const int tile = blockIdx.x * 4 + (threadIdx.x >> 5);
  if (tile >= __ldg(n_tiles_ptr)) return;
  const int* cm = col_mol + (size_t)tile * nt;
  int n_before = 0;
  for (int w = 0; w < 4; ++w) {
    const int c = w * 32 + lane;
    bool end = false;
    int m = -1;
    if (c < nt) {
      m = __ldg(cm + c);
      end = c == nt - 1 || __ldg(cm + c + 1) != m;
    }
    const unsigned mask = __ballot_sync(0xffffffffu, end);
    // mult = D if every Z offset m * D fits 31 bits (the epilogue then adds it to a 64-bit base), else 1
    if (end) run_mol[(size_t)tile * nt + n_before + __popc(mask & ((1u << lane) - 1u))] = m < 0 ? -1 : m * mult;
    if (lane == 0) end_mask[(size_t)tile * 4 + w] = mask;
    n_before += __popc(mask);
  }
}

// ---------------------------------------------------------------------------------------------------
// 2. X tiles: block = one tile of nt columns.  Xh / Xl [tile][kb][nt][64 halves] swizzled; inv_scale[tile].
// ---------------------------------------------------------------------------------------------------
static __global__ void __launch_bounds__(256)
fm_prep_x_kernel(const float* __restrict__ x, const int* __restrict__ col_atom, const int* __restrict__ n_tiles_ptr,
                 int d, int nt, __half* __restrict__ Xh, __half* __restrict__ Xl, float* __restrict__ inv_scale) {
  __shared__ float red[8];
  __shared__ int atom_s[128];
  const int tile = blockIdx.x;
  if (tile >= __ldg(n_tiles_ptr)) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x < nt) atom_s[threadIdx.x] = __ldg(col_atom + (size_t)tile * nt + threadIdx.x);
  __syncthreads();
  const int d4 = d / 4;
  float amax = 0.f;
  for (int item = threadIdx.x; item < nt * d4; item += 256) {
    const int a = atom_s[item / d4];
    if (a >= 0) {
      const float4 v = __ldg(reinterpret_cast<const float4*>(x + (size_t)a * d) + item % d4);
      amax = fmaxf(amax, fmaxf(fmaxf(fabsf(v.x), fabsf(v.y)), fmaxf(fabsf(v.z), fabsf(v.w))));
    }
  }
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, m));
  if (lane == 0) red[warp] = amax;
  __syncthreads();
  amax = red[0];
#pragma unroll
  for (int w = 1; w < 8; ++w) amax = fmaxf(amax, red[w]);
  int sh = 9 - ((int)((__float_as_uint(amax) >> 23) & 0xffu) - 127);       // amax * s in [2^9, 2^10)
  if (amax == 0.f) sh = 0;
  sh = sh < -100 ? -100 : (sh > 100 ? 100 : sh);
  const float s = __uint_as_float((uint32_t)(127 + sh) << 23);
  if (threadIdx.x == 0) inv_scale[tile] = __uint_as_float((uint32_t)(127 - sh) << 23);
  const int kKB = d / kKBlk;
  // one thread = one 16-byte chunk (8 inputs) of one column
  for (int item = threadIdx.x; item < nt * (d / 8); item += 256) {
    const int col = item / (d / 8), ck = item % (d / 8);
    const int kb = ck >> 3, ch = ck & 7;
    const int a = atom_s[col];
    __half h[8], l[8];
    if (a >= 0) {
      const float4 v0 = __ldg(reinterpret_cast<const float4*>(x + (size_t)a * d + ck * 8));
      const float4 v1 = __ldg(reinterpret_cast<const float4*>(x + (size_t)a * d + ck * 8) + 1);
      const float f[8] = {v0.x * s, v0.y * s, v0.z * s, v0.w * s, v1.x * s, v1.y * s, v1.z * s, v1.w * s};
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        h[u] = __float2half_rn(f[u]);
        l[u] = __float2half_rn(f[u] - __half2float(h[u]));
      }
    } else {
#pragma unroll
      for (int u = 0; u < 8; ++u) h[u] = l[u] = __float2half_rn(0.f);
    }
    const size_t row = ((size_t)tile * kKB + kb) * nt + col;
    const size_t o = row * 64 + (size_t)((ch ^ (int)(col & 7)) << 3);
    *reinterpret_cast<uint4*>(Xh + o) = *reinterpret_cast<const uint4*>(h);
    *reinterpret_cast<uint4*>(Xl + o) = *reinterpret_cast<const uint4*>(l);
  }
}

// ---------------------------------------------------------------------------------------------------
// 3. Dense W (RFF): per-element power-of-two scale, hi / lo tiles [e][ft][kb][128][64] swizzled.
// ---------------------------------------------------------------------------------------------------
static __global__ void __launch_bounds__(256)
fm_w_amax_kernel(const float* __restrict__ W, size_t per_elem, unsigned* __restrict__ amax_bits) {
  const int e = blockIdx.y;
  float amax = 0.f;
  for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < per_elem; i += (size_t)gridDim.x * 256)
    amax = fmaxf(amax, fabsf(__ldg(W + (size_t)e * per_elem + i)));
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, m));
  if ((threadIdx.x & 31) == 0) atomicMax(amax_bits + e, __float_as_uint(amax));   // non-negative floats order as uints
}

// block = (feature tile ft, element e); thread = 16-byte chunk of one row
static __global__ void __launch_bounds__(256)
fm_prep_w_kernel(const float* __restrict__ W, const unsigned* __restrict__ amax_bits, int D, int d,
                 __half* __restrict__ Wh, __half* __restrict__ Wl, float* __restrict__ inv_wscale) {
  const int ft = blockIdx.x, e = blockIdx.y, n_ft = (D + kTile - 1) / kTile, kKB = d / kKBlk;
  const float amax = __uint_as_float(__ldg(amax_bits + e));
  int sh = 9 - ((int)((__float_as_uint(amax) >> 23) & 0xffu) - 127);
  if (amax == 0.f) sh = 0;
  sh = sh < -100 ? -100 : (sh > 100 ? 100 : sh);
  const float s = __uint_as_float((uint32_t)(127 + sh) << 23);
  if (ft == 0 && threadIdx.x == 0) inv_wscale[e] = __uint_as_float((uint32_t)(127 - sh) << 23);
  for (int item = threadIdx.x; item < kTile * (d / 8); item += 256) {
    const int row = item / (d / 8), ck = item % (d / 8);
    const int kb = ck >> 3, ch = ck & 7;
    const int l = ft * kTile + row;
    __half h[8], lo[8];
    if (l < D) {
      const float* src = W + ((size_t)e * D + l) * d + ck * 8;
      const float4 v0 = __ldg(reinterpret_cast<const float4*>(src)), v1 = __ldg(reinterpret_cast<const float4*>(src) + 1);
      const float f[8] = {v0.x * s, v0.y * s, v0.z * s, v0.w * s, v1.x * s, v1.y * s, v1.z * s, v1.w * s};
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        h[u] = __float2half_rn(f[u]);
        lo[u] = __float2half_rn(f[u] - __half2float(h[u]));
      }
    } else {
#pragma unroll
      for (int u = 0; u < 8; ++u) h[u] = lo[u] = __float2half_rn(0.f);
    }
    const size_t tile = ((size_t)e * n_ft + ft) * kKB + kb;
    const size_t o = tile * (kTile * kKBlk) + (size_t)row * 64 + (size_t)((ch ^ (row & 7)) << 3);
    *reinterpret_cast<uint4*>(Wh + o) = *reinterpret_cast<const uint4*>(h);
    *reinterpret_cast<uint4*>(Wl + o) = *reinterpret_cast<const uint4*>(lo);
  }
}

// ---------------------------------------------------------------------------------------------------
// 4. The tcgen05 kernel.
// ---------------------------------------------------------------------------------------------------
template <int D_, bool kRff>
struct FmCfg {
  static constexpr int d = D_;
  static constexpr int kKB = D_ / kKBlk;
  static constexpr int kParts = kRff ? 2 : 1;                                  // W parts in shared memory (hi, lo)
  static constexpr int kCtas = D_ <= 128 ? 2 : 1;                              // CTAs per SM
  static constexpr int kG = (D_ <= 128 ? 4 : 2) / kParts / kCtas;              // 128-feature tiles per task
  static constexpr int kNT = fm_nt(D_);                                        // atoms per tile
  static constexpr int kStages = kCtas == 2 ? 2 : (D_ <= 128 ? 4 : 3);
  static constexpr int kTmemCols = 512 / kCtas;
  static constexpr int kTBufRaw = kTmemCols / (kG * kNT);
  static constexpr int kTBuf = kTBufRaw > 4 ? 4 : kTBufRaw;
  static constexpr uint32_t kABytes = kParts * kG * kKB * kTileBytes;          // 128 KB
  static constexpr uint32_t kStageBytes = 2 * kNT * 128;                       // hi + lo tile of one k-block
  static constexpr int kEpiWarps = 16;                                         // 4 groups of 4 TMEM lane quarters
  static constexpr int kTPW = kG >= 4 ? kG / 4 : 1;                            // feature tiles per epilogue warp
  static constexpr int kColSplit = kG >= 4 ? 1 : 4 / kG;                       // groups that share a tile split its columns
  static constexpr int kThreads = 64 + 32 * kEpiWarps;
  static constexpr uint32_t kSmem = kABytes + kStages * kStageBytes + 512 + 1024;
  static_assert(kTBuf >= 2, "TMEM double buffering");
  static_assert((kNT / kColSplit) % 8 == 0, "column pieces of 8");
};

template <int D_, bool kRff>
__global__ void __launch_bounds__(FmCfg<D_, kRff>::kThreads, FmCfg<D_, kRff>::kCtas)
featmap_mma_kernel(const int* __restrict__ tile_elem, const int* __restrict__ n_tiles_ptr,
                   const uint32_t* __restrict__ end_mask, const int* __restrict__ run_mol, int D, int n_ft, float c, const float* __restrict__ c_elem,
                   float nrm, const __half* __restrict__ Wh, const __half* __restrict__ Wl,
                   const __half* __restrict__ Xh, const __half* __restrict__ Xl, const float* __restrict__ inv_scale,
                   const float* __restrict__ bias, int n_chunks, int run_stride, float* __restrict__ Z) {
  using C = FmCfg<D_, kRff>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint8_t* a_smem = smem;                        // [part][g][kb] tiles of 16 KB
  uint8_t* b_smem = smem + C::kABytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(b_smem + C::kStages * C::kStageBytes);
  uint64_t* a_full = bars;                       // [kKB]
  uint64_t* a_empty = bars + C::kKB;             // [kKB]
  uint64_t* b_full = bars + 2 * C::kKB;          // [kStages]
  uint64_t* b_empty = b_full + C::kStages;       // [kStages]
  uint64_t* t_full = b_empty + C::kStages;       // [kTBuf]
  uint64_t* t_empty = t_full + C::kTBuf;         // [kTBuf]
  uint32_t* tmem_ptr_smem = reinterpret_cast<uint32_t*>(t_empty + C::kTBuf);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_fg = (n_ft + C::kG - 1) / C::kG;              // feature groups
  const int n_tiles = __ldg(n_tiles_ptr);
  const long long n_tasks = (long long)n_chunks * n_fg;

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::kKB; ++i) { mbar_init(&a_full[i], 1); mbar_init(&a_empty[i], 1); }
    for (int i = 0; i < C::kStages; ++i) { mbar_init(&b_full[i], 1); mbar_init(&b_empty[i], 1); }
    for (int i = 0; i < C::kTBuf; ++i) { mbar_init(&t_full[i], 1); mbar_init(&t_empty[i], C::kEpiWarps); }
    fence_mbarrier_init();
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_ptr_smem)), "n"(C::kTmemCols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  const uint32_t tmem_base = *tmem_ptr_smem;

  if (warp == 0) {
    // ===================== producer =====================
    if (lane == 0) {
      uint32_t n_a = 0, n_b = 0;
      for (long long task = blockIdx.x; task < n_tasks; task += gridDim.x) {
        const int fg = (int)(task % n_fg), ch = (int)(task / n_fg);
        const int t_begin = ch * kFmChunkTiles;
        const int t_end = t_begin + kFmChunkTiles < n_tiles ? t_begin + kFmChunkTiles : n_tiles;
        const int g0 = fg * C::kG;
        const int n_g = n_ft - g0 < C::kG ? n_ft - g0 : C::kG;
        int e_prev = -1;
        for (int tile = t_begin; tile < t_end; ++tile) {
          const int e = __ldg(tile_elem + tile);
          if (e != e_prev) {
#pragma unroll 1
            for (int kb = 0; kb < C::kKB; ++kb) {
              if (n_a > 0) mbar_wait(&a_empty[kb], (n_a - 1) & 1);
              mbar_expect_tx(&a_full[kb], (uint32_t)(C::kParts * n_g) * kTileBytes);
              for (int g = 0; g < n_g; ++g) {
                const size_t src = (((size_t)e * n_ft + g0 + g) * C::kKB + kb) * (size_t)(kTile * kKBlk);
                bulk_copy_g2s(a_smem + (g * C::kKB + kb) * kTileBytes, Wh + src, kTileBytes, &a_full[kb]);
                if (kRff)
                  bulk_copy_g2s(a_smem + ((C::kG + g) * C::kKB + kb) * kTileBytes, Wl + src, kTileBytes, &a_full[kb]);
              }
            }
            ++n_a;
            e_prev = e;
          }
          for (int kb = 0; kb < C::kKB; ++kb, ++n_b) {
            const uint32_t st = n_b % C::kStages, use = n_b / C::kStages;
            if (use > 0) mbar_wait(&b_empty[st], (use - 1) & 1);
            constexpr uint32_t bytes = (uint32_t)C::kNT * 128;
            mbar_expect_tx(&b_full[st], 2 * bytes);
            const size_t row = ((size_t)tile * C::kKB + kb) * C::kNT;
            uint8_t* dst = b_smem + st * C::kStageBytes;
            bulk_copy_g2s(dst, Xh + row * 64, bytes, &b_full[st]);
            bulk_copy_g2s(dst + bytes, Xl + row * 64, bytes, &b_full[st]);
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer: the whole warp runs the loop, one elected lane issues =====================
    const bool leader = elect_one_sync();
    const uint32_t tmem_base_u = __shfl_sync(0xffffffffu, tmem_base, 0);
    uint64_t a_desc[C::kParts][C::kG][C::kKB], b_desc[C::kStages];
#pragma unroll
    for (int pt = 0; pt < C::kParts; ++pt)
#pragma unroll
      for (int g = 0; g < C::kG; ++g)
#pragma unroll
        for (int kb = 0; kb < C::kKB; ++kb)
          a_desc[pt][g][kb] = make_kmajor_sw128_desc(smem_u32(a_smem + ((pt * C::kG + g) * C::kKB + kb) * kTileBytes));
#pragma unroll
    for (int st = 0; st < C::kStages; ++st) b_desc[st] = make_kmajor_sw128_desc(smem_u32(b_smem + st * C::kStageBytes));
    constexpr uint64_t kLoOff = (uint64_t)((C::kNT * 128) >> 4);
    constexpr uint32_t idesc = (1u << 4) | ((uint32_t)(C::kNT >> 3) << 17) | ((uint32_t)(kTile >> 4) << 24);
    uint32_t n_a = 0, n_b = 0, n_t = 0;
    for (long long task = blockIdx.x; task < n_tasks; task += gridDim.x) {
      const int fg = (int)(task % n_fg), ch = (int)(task / n_fg);
      const int t_begin = ch * kFmChunkTiles;
      const int t_end = t_begin + kFmChunkTiles < n_tiles ? t_begin + kFmChunkTiles : n_tiles;
      const int g0 = fg * C::kG;
      const int n_g = n_ft - g0 < C::kG ? n_ft - g0 : C::kG;
      int e_prev = -1;
      int e_next = t_begin < t_end ? __shfl_sync(0xffffffffu, __ldg(tile_elem + t_begin), 0) : -1;
      for (int tile = t_begin; tile < t_end; ++tile, ++n_t) {
        const int e = e_next;
        e_next = (tile + 1 < t_end) ? __shfl_sync(0xffffffffu, __ldg(tile_elem + tile + 1), 0) : -1;
        const bool first_of_run = e != e_prev;
        if (first_of_run) { ++n_a; e_prev = e; }
        const bool last_of_run = e_next != e;
        const uint32_t tb = n_t % C::kTBuf, tuse = n_t / C::kTBuf;
        if (tuse > 0) mbar_wait(&t_empty[tb], (tuse - 1) & 1);
        tcgen05_fence_after();
        const uint32_t tmem_tile = tmem_base_u + tb * (C::kG * C::kNT);
#pragma unroll
        for (int kb = 0; kb < C::kKB; ++kb, ++n_b) {
          const uint32_t st = n_b % C::kStages;
          if (first_of_run) mbar_wait(&a_full[kb], (n_a - 1) & 1);
          mbar_wait(&b_full[st], (n_b / C::kStages) & 1);
          tcgen05_fence_after();
          uint64_t b_hi = b_desc[0];
#pragma unroll
          for (int q = 1; q < C::kStages; ++q) b_hi = (st == (uint32_t)q) ? b_desc[q] : b_hi;
          if (leader) {
#pragma unroll
            for (int kk = 0; kk < kKBlk / 16; ++kk) {
              const uint64_t adv = (uint64_t)((kk * 32) >> 4);
              const uint32_t acc0 = (kb > 0 || kk > 0) ? 1u : 0u;
              // small terms first; consecutive MMAs go to different accumulators
#pragma unroll
              for (int g = 0; g < C::kG; ++g)
                if (g < n_g) umma<true>(tmem_tile + g * C::kNT, a_desc[0][g][kb] + adv, b_hi + kLoOff + adv, idesc, acc0);
              if (kRff) {
#pragma unroll
                for (int g = 0; g < C::kG; ++g)
                  if (g < n_g)
                    umma<true>(tmem_tile + g * C::kNT, a_desc[C::kParts - 1][g][kb] + adv, b_hi + adv, idesc, 1u);
              }
#pragma unroll
              for (int g = 0; g < C::kG; ++g)
                if (g < n_g) umma<true>(tmem_tile + g * C::kNT, a_desc[0][g][kb] + adv, b_hi + adv, idesc, 1u);
            }
            tcgen05_commit(&b_empty[st]);
            if (last_of_run) tcgen05_commit(&a_empty[kb]);
          }
          __syncwarp();
        }
        if (leader) tcgen05_commit(&t_full[tb]);
        __syncwarp();
      }
    }
  } else {
    // ===================== epilogue warps: thread = output feature =====================
    // 16 warps = 4 groups x 4 TMEM lane quarters.  A group owns kTPW feature tiles (all columns) or, when there are
    // fewer tiles than groups, a range of columns of one tile.  Per column: FFMA, cos, FADD and one bit test; per run of
    // columns of one molecule: one load of the molecule index and one fp32 reduction into Z per owned tile.
    const int warp_u = __shfl_sync(0xffffffffu, warp, 0);   // provably uniform: the column bit tests become uniform branches
    const int quarter = warp_u & 3;             // TMEM lanes [32 q, 32 q + 32)
    const int grp = (warp_u - 2) >> 2;          // 0..3
    const int row = quarter * 32 + lane;
    constexpr int kCols = C::kNT / C::kColSplit;
    const int col_lo = (grp % C::kColSplit) * kCols;
    const int t_lo = C::kColSplit > 1 ? grp / C::kColSplit : grp * C::kTPW;
    uint32_t n_t = 0;
    for (long long task = blockIdx.x; task < n_tasks; task += gridDim.x) {
      const int fg = (int)(task % n_fg), ch = (int)(task / n_fg);
      const int t_begin = ch * kFmChunkTiles;
      const int t_end = t_begin + kFmChunkTiles < n_tiles ? t_begin + kFmChunkTiles : n_tiles;
      float* zf[C::kTPW];                       // Z + feature (features past D: a column of the last valid feature, never added)
      bool live[C::kTPW];
      int feat[C::kTPW];
      float acc[C::kTPW], bv[C::kTPW];
#pragma unroll
      for (int w = 0; w < C::kTPW; ++w) {
        feat[w] = (fg * C::kG + t_lo + w) * kTile + row;
        live[w] = feat[w] < D;
        zf[w] = Z + (live[w] ? feat[w] : 0);
        acc[w] = 0.f;
        bv[w] = 0.f;
      }
      int e_prev = -1;
      float ce = c;
      for (int tile = t_begin; tile < t_end; ++tile, ++n_t) {
        const int e = __shfl_sync(0xffffffffu, __ldg(tile_elem + tile), 0);
        if (e != e_prev) {
#pragma unroll
          for (int w = 0; w < C::kTPW; ++w) bv[w] = live[w] ? __ldg(bias + (size_t)e * D + feat[w]) : 0.f;
          if (kRff) ce = __ldg(c_elem + e);
          e_prev = e;
        }
        const float sc = ce * __ldg(inv_scale + tile);
        // run ends of this tile (uniform: made provably so with a shuffle, so that the bit tests are uniform branches)
        const uint32_t em0 = __shfl_sync(0xffffffffu, __ldg(end_mask + (size_t)tile * 4 + 0), 0);
        const uint32_t em1 = __shfl_sync(0xffffffffu, __ldg(end_mask + (size_t)tile * 4 + 1), 0);
        const uint32_t em2 = __shfl_sync(0xffffffffu, __ldg(end_mask + (size_t)tile * 4 + 2), 0);
        const unsigned long long em01 = (unsigned long long)em0 | ((unsigned long long)em1 << 32);
        // index of the run that contains column col_lo = number of run ends before it
        int run = col_lo >= 64 ? __popcll(em01) + __popc(em2 & ((1u << (col_lo - 64)) - 1u))
                               : __popcll(em01 & ((1ull << col_lo) - 1ull));
        const int* rm = run_mol + (size_t)tile * C::kNT;
        const uint32_t tb = n_t % C::kTBuf;
        mbar_wait(&t_full[tb], (n_t / C::kTBuf) & 1);
        tcgen05_fence_after();
        constexpr int kP = kCols % 16 == 0 ? 16 : 8;     // columns per TMEM load
#pragma unroll 1
        for (int r0 = 0; r0 < kCols; r0 += kP) {
          uint32_t u[C::kTPW][kP];
#pragma unroll
          for (int w = 0; w < C::kTPW; ++w) {
            const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16) + tb * (C::kG * C::kNT) +
                                   (t_lo + w) * C::kNT + col_lo + r0;
            if constexpr (kP == 16) {
              tmem_ld_32x32b_x16(taddr, u[w]);
            } else {
              tmem_ld_32x32b_x8(taddr, u[w]);
            }
          }
          const int c0 = col_lo + r0;
          const uint32_t true_ends = (c0 >= 64 ? em2 >> (c0 - 64) : (uint32_t)(em01 >> c0)) & ((1u << kP) - 1u);
          const uint32_t bits = true_ends | (r0 + kP == kCols ? 1u << (kP - 1) : 0u);   // the group's last column closes its run
          tmem_ld_wait();
          // all cos of the piece first (independent: the MUFU latencies overlap), then the sequential run logic
          float z[C::kTPW][kP];
#pragma unroll
          for (int w = 0; w < C::kTPW; ++w)
#pragma unroll
            for (int r = 0; r < kP; ++r) z[w][r] = __cosf(fmaf(sc, __uint_as_float(u[w][r]), bv[w]));
#pragma unroll
          for (int r = 0; r < kP; ++r) {
#pragma unroll
            for (int w = 0; w < C::kTPW; ++w) acc[w] += z[w][r];
            if (bits & (1u << r)) {
              const int m = __ldg(rm + run);
              if (m >= 0) {
#pragma unroll
                for (int w = 0; w < C::kTPW; ++w)
                  if (live[w]) atomicAdd(zf[w] + (size_t)(uint32_t)m * (size_t)(uint32_t)run_stride, nrm * acc[w]);
              }
#pragma unroll
              for (int w = 0; w < C::kTPW; ++w) acc[w] = 0.f;
              run += (true_ends >> r) & 1u;
            }
          }
        }
        tcgen05_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&t_empty[tb]);
      }
    }
  }

  tcgen05_fence_before();
  __syncthreads();
  if (warp == 2) {
    tcgen05_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(C::kTmemCols) : "memory");
  }
}

// ---------------------------------------------------------------------------------------------------
// Host side
// ---------------------------------------------------------------------------------------------------
bool featmap_mma_supported(int d, int n_elem) { return (d == 128 || d == 256) && n_elem >= 1 && n_elem <= kFmMaxElem; }

static size_t fm_groups(int64_t n_atoms) {
  const size_t n_blk = (size_t)((n_atoms + kFmSortThreads - 1) / kFmSortThreads);
  return (n_blk + kFmGrpBlks - 1) / kFmGrpBlks;
}
static size_t fm_tiles_max(int64_t n_atoms, int d, int n_elem) {
  return (size_t)((n_atoms + fm_nt(d) - 1) / fm_nt(d)) + fm_groups(n_atoms) * n_elem;
}

// bytes of everything but the W tables
size_t featmap_mma_scratch_bytes(int d, int n_elem, int64_t n_atoms) {
  const size_t tiles = fm_tiles_max(n_atoms, d, n_elem), cols = tiles * fm_nt(d);
  const size_t n_blk = (size_t)((n_atoms + kFmSortThreads - 1) / kFmSortThreads);
  return 2 * align_up(cols * (size_t)d * sizeof(__half), 256) + 3 * align_up(cols * sizeof(int), 256) +
         2 * align_up(tiles * sizeof(int), 256) + align_up(tiles * 16, 256) + 2 * align_up(n_blk * n_elem * sizeof(int) + 4, 256) +
         2 * align_up((fm_groups(n_atoms) * n_elem + 1) * sizeof(int), 256) + 16 * 256;
}
size_t featmap_mma_w_bytes(int d, int D, int n_elem, bool rff) {
  const size_t n_ft = (size_t)(D + kTile - 1) / kTile;
  return (rff ? 2 : 1) * align_up((size_t)n_elem * n_ft * kTile * d * sizeof(__half), 256) +
         (rff ? 2 * align_up((size_t)n_elem * sizeof(float), 256) : 0) + 4 * 256;
}

template <int D_, bool kRff>
static int launch_featmap(int n_elem, int D, float c, const float* c_elem, const __half* Wh, const __half* Wl,
                          const float* bias, const float* x, const int32_t* elem, const int32_t* mol_off,
                          int64_t n_atoms, int32_t n_mol, float* Z, Carver& ws, cudaStream_t st) {
  using C = FmCfg<D_, kRff>;
  constexpr int nt = C::kNT;
  const size_t tiles = fm_tiles_max(n_atoms, D_, n_elem), cols = tiles * nt;
  const int n_blk = (int)((n_atoms + kFmSortThreads - 1) / kFmSortThreads);
  __half* Xh = ws.take<__half>(cols * D_);
  __half* Xl = ws.take<__half>(cols * D_);
  int* col_atom = ws.take<int>(cols);
  int* col_mol = ws.take<int>(cols);
  int* tile_elem = ws.take<int>(tiles);
  float* inv_scale = ws.take<float>(tiles);
  uint32_t* end_mask = ws.take<uint32_t>(tiles * 4);
  int* run_mol = ws.take<int>(cols);
  int* blk_cnt = ws.take<int>((size_t)n_blk * n_elem + 1);
  int* blk_off = ws.take<int>((size_t)n_blk * n_elem + 1);
  const int n_grp = (int)fm_groups(n_atoms), n_keys = n_grp * n_elem;
  int* key_cnt = ws.take<int>((size_t)n_keys + 1);
  int* key_tile0 = ws.take<int>((size_t)n_keys + 1);
  if (!ws.fits()) return QMLL_ERR_WORKSPACE;
  QMLL_CUDA_TRY(cudaMemsetAsync(Z, 0, (size_t)n_mol * D * sizeof(float), st));
  QMLL_CUDA_TRY(cudaMemsetAsync(col_atom, 0xff, cols * sizeof(int), st));
  QMLL_CUDA_TRY(cudaMemsetAsync(col_mol, 0xff, cols * sizeof(int), st));
  fm_block_count_kernel<<<n_blk, kFmSortThreads, 0, st>>>(elem, n_atoms, n_elem, blk_cnt);
  QMLL_LAUNCH_CHECK("fm_block_count_kernel");
  fm_group_scan_kernel<<<(n_keys + 255) / 256, 256, 0, st>>>(blk_cnt, n_blk, n_grp, n_elem, blk_off, key_cnt);
  QMLL_LAUNCH_CHECK("fm_group_scan_kernel");
  fm_tile_scan_kernel<<<1, 32, 0, st>>>(key_cnt, n_keys, nt, key_tile0);
  QMLL_LAUNCH_CHECK("fm_tile_scan_kernel");
  fm_place_kernel<<<n_blk, kFmSortThreads, 0, st>>>(elem, mol_off, n_atoms, n_mol, n_elem, nt, blk_off, key_tile0,
                                                    col_atom, col_mol);
  QMLL_LAUNCH_CHECK("fm_place_kernel");
  fm_tile_elem_kernel<<<(unsigned)((tiles + 255) / 256), 256, 0, st>>>(key_tile0, n_keys, n_elem, (int)tiles, tile_elem);
  QMLL_LAUNCH_CHECK("fm_tile_elem_kernel");
  const bool small = (long long)n_mol * D < 0x7fffffffLL;      // every Z offset fits 31 bits: the run table holds m * D
  fm_runs_kernel<<<(unsigned)((tiles + 3) / 4), 128, 0, st>>>(col_mol, key_tile0 + n_keys, nt, small ? D : 1, end_mask,
                                                              run_mol);
  QMLL_LAUNCH_CHECK("fm_runs_kernel");
  fm_prep_x_kernel<<<(unsigned)tiles, 256, 0, st>>>(x, col_atom, key_tile0 + n_keys, D_, nt, Xh, Xl, inv_scale);
  QMLL_LAUNCH_CHECK("fm_prep_x_kernel");
  auto kern = featmap_mma_kernel<D_, kRff>;
  QMLL_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::kSmem));
  const int n_ft = (D + kTile - 1) / kTile;
  const int n_chunks = (int)((tiles + kFmChunkTiles - 1) / kFmChunkTiles);
  const long long n_tasks = (long long)n_chunks * ((n_ft + C::kG - 1) / C::kG);
  const int grid = (int)(n_tasks < device_sm_count() * C::kCtas ? n_tasks : device_sm_count() * C::kCtas);
  const float nrm = (float)sqrt(2.0 / (double)D);
  kern<<<grid, C::kThreads, C::kSmem, st>>>(tile_elem, key_tile0 + n_keys, end_mask, run_mol, D, n_ft, c, c_elem, nrm, Wh, Wl, Xh, Xl,
                                            inv_scale, bias, n_chunks, small ? 1 : D, Z);
  QMLL_LAUNCH_CHECK("featmap_mma_kernel");
  return QMLL_OK;
}

// SORF: W16 = the fp16 table of sorf_mma_build_w
int featmap_sorf_forward_mma(const SorfProblem& pr, const void* W16, float* Z, Carver& ws, cudaStream_t st) {
  const qmll_sorf_params* p = pr.p;
  if (pr.n_mol == 0) return QMLL_OK;
  if (pr.n_atoms == 0) {
    QMLL_CUDA_TRY(cudaMemsetAsync(Z, 0, (size_t)pr.n_mol * p->D * sizeof(float), st));
    return QMLL_OK;
  }
  const float c = (float)(sqrt((double)p->d) / (double)p->sigma * pow((double)p->d, -0.5 * p->n_transform));
  if (p->d == 128)
    return launch_featmap<128, false>(p->n_elem, p->D, c, nullptr, (const __half*)W16, nullptr, p->bias, pr.x, pr.elem,
                                      pr.mol_off, pr.n_atoms, pr.n_mol, Z, ws, st);
  if (p->d == 256)
    return launch_featmap<256, false>(p->n_elem, p->D, c, nullptr, (const __half*)W16, nullptr, p->bias, pr.x, pr.elem,
                                      pr.mol_off, pr.n_atoms, pr.n_mol, Z, ws, st);
  return QMLL_ERR_UNSUPPORTED;
}

// RFF: dense W [n_elem, D, d] fp32
int featmap_rff_forward(const float* W, const float* bias, int d, int D, int n_elem, const float* x, const int32_t* elem,
                        const int32_t* mol_off, int64_t n_atoms, int32_t n_mol, float* Z, Carver& ws, cudaStream_t st) {
  if (n_mol == 0) return QMLL_OK;
  if (n_atoms == 0) {
    QMLL_CUDA_TRY(cudaMemsetAsync(Z, 0, (size_t)n_mol * D * sizeof(float), st));
    return QMLL_OK;
  }
  const size_t n_ft = (size_t)(D + kTile - 1) / kTile;
  __half* Wh = ws.take<__half>((size_t)n_elem * n_ft * kTile * d);
  __half* Wl = ws.take<__half>((size_t)n_elem * n_ft * kTile * d);
  float* inv_wscale = ws.take<float>(n_elem);
  unsigned* amax_bits = ws.take<unsigned>(n_elem);
  if (!ws.fits()) return QMLL_ERR_WORKSPACE;
  QMLL_CUDA_TRY(cudaMemsetAsync(amax_bits, 0, n_elem * sizeof(unsigned), st));
  fm_w_amax_kernel<<<dim3(64, n_elem), 256, 0, st>>>(W, (size_t)D * d, amax_bits);
  QMLL_LAUNCH_CHECK("fm_w_amax_kernel");
  fm_prep_w_kernel<<<dim3((unsigned)n_ft, n_elem), 256, 0, st>>>(W, amax_bits, D, d, Wh, Wl, inv_wscale);
  QMLL_LAUNCH_CHECK("fm_prep_w_kernel");
  if (d == 128)
    return launch_featmap<128, true>(n_elem, D, 1.f, inv_wscale, Wh, Wl, bias, x, elem, mol_off, n_atoms, n_mol, Z, ws, st);
  if (d == 256)
    return launch_featmap<256, true>(n_elem, D, 1.f, inv_wscale, Wh, Wl, bias, x, elem, mol_off, n_atoms, n_mol, Z, ws, st);
  return QMLL_ERR_UNSUPPORTED;
}

}  // namespace qmll
