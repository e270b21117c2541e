// sorf_mma.cu -- force rows (step a7: G = -dZ/dr, eq. 17) on the tensor cores.
//
// The SORF map of one stack is LINEAR: (H S_T ... H S_1) = W_{e,s}, a d x d matrix of small integers, and the
// force rows apply it to 3 n^2 gradient columns per molecule -- a dense contraction with the same matrix for every
// column of the same (element, stack).  The register FWHT needs d log2(d) T adds + d T sign flips per column and is
// bound by fp32/integer issue (62 % of the measured FADD peak at best); the explicit product needs d^2 MACs but runs
// on tcgen05 at ~30x the rate, so it is 2.5-3.5x faster for d = 128 / 256:
//   1. build_w_kernel:  W_{e,s} for every (element, stack) by pushing the d unit vectors through the SAME
//      register chain the other kernels use (exact: integers below 2^24), stored as fp16.  |W_ij| <= d^(3/2) (Cauchy-
//      Schwarz on the orthogonal rows of H S H) and all entries are even for T = 3, so fp16 holds them EXACTLY for
//      d <= 256 (d = 128: <= 1448 < 2048; d = 256: even integers <= 4096); T <= 2 gives |W_ij| <= d.
//   2. prep_columns_kernel:  gradient block of atom I, [d, 3n] fp32 -> columns split into fp16 hi + lo parts (22
//      significant bits, the same split as the normal equations) with one power-of-two scale per atom block,
//      k-block-major and pre-swizzled, so that a tile is one contiguous bulk copy.
//   3. sorf_rows_mma_kernel:  persistent, warp-specialised (bulk-copy producer / MMA issuer / epilogue warps).  Task =
//      (molecule, stack): for every atom I:  U_I = W_{e_I,s} X_I  (tcgen05.mma kind::f16, hi and lo passes, fp32
//      accumulate in TMEM), and the epilogue adds  c * zs_I[l] * U_I[l, r]  into 3n register accumulators per thread
//      (thread = output feature l); the finished [3n, d] block of G is written once, coalesced along l.
// The result is the same linear map applied to the same inputs: parity against the FP64 oracle is unchanged.
#include <cuda_fp16.h>

#include "sorf_kernels.cuh"
#include "tcgen05_utils.cuh"

namespace qmll {


// ---------------------------------------------------------------------------------------------------
// 1. W table.  Warp = (element e, stack group sg, input index j); lanes = stacks (as everywhere).  The unit vector
//    e_j goes through the chain; lane (sl, p) then holds column j of W_{e,s} for outputs p*E .. p*E+E-1.
//    W16 tile index: ((e*n_s + s)*kMT + mt)*kKB + kb, tile = [128 outputs][64 inputs] halves, swizzled.
// ---------------------------------------------------------------------------------------------------
template <typename S>
__global__ void __launch_bounds__(kFwdThreads, (S::E >= 128 ? 3 : 4))
build_w_kernel(const uint32_t* __restrict__ sign_bits, int n_elem, int n_s, int n_sg, int T,
               __half* __restrict__ W16) {
  constexpr int kMT = S::d / kTile, kKB = S::d / kKBlk;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long task = (long long)blockIdx.x * (kFwdThreads / kWarp) + warp;
  if (task >= (long long)n_elem * n_sg * S::d) return;
  const int j = (int)(task % S::d);
  const int sg = (int)((task / S::d) % n_sg);
  const int e = (int)(task / ((long long)S::d * n_sg));
  const int p = lane % S::P, sl = lane / S::P;
  const int s = sg * S::SPW + sl;
  f32x2 v[S::E2];
#pragma unroll
  for (int q = 0; q < S::E2; ++q) {
    const int m = p * S::E + 2 * q;
    v[q] = pk(m == j ? 1.f : 0.f, m + 1 == j ? 1.f : 0.f);
  }
  chain_forward<S>(v, sign_bits, e, T, n_sg, sg, lane);
  if (s >= n_s) return;
  const int kb = j / kKBlk, jj = j % kKBlk;
#pragma unroll
  for (int q = 0; q < S::E2; ++q) {
    float a, b;
    upk(v[q], a, b);
    const int i = p * S::E + 2 * q;                       // output index (even), i + 1 is the odd one
    const int mt = i / kTile, row = i % kTile;
    __half* tile = W16 + ((((size_t)e * n_s + s) * kMT + mt) * kKB + kb) * (size_t)(kTile * kKBlk);
    tile[swz_half_index(row, jj)] = __float2half_rn(a);
    tile[swz_half_index(row + 1, jj)] = __float2half_rn(b);
  }
}

// ---------------------------------------------------------------------------------------------------
// 2. Column preparation.  xoff[M] = first 128-byte row of molecule M in Xh / Xl; the block of atom I (local) holds
//    kKB sub-blocks of Npad = roundup16(3n) rows: row = xoff[M] + (I*kKB + kb)*Npad + col, 64 halves per row
//    (inputs 64 kb .. 64 kb + 63 of column col), swizzled; rows col >= 3n are zero.
// ---------------------------------------------------------------------------------------------------
static __global__ void __launch_bounds__(1024)
x_offsets_kernel(const int32_t* __restrict__ mol_off, int n_mol, int kKB, long long* __restrict__ xoff) {
  __shared__ long long part[1024];
  __shared__ long long carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int base = 0; base < n_mol; base += 1024) {
    const int M = base + threadIdx.x;
    long long cnt = 0;
    if (M < n_mol) {
      const long long n = __ldg(mol_off + M + 1) - __ldg(mol_off + M);
      cnt = n * kKB * ((3 * n + 15) / 16 * 16);
    }
    part[threadIdx.x] = cnt;
    __syncthreads();
    for (int off = 1; off < 1024; off <<= 1) {
      const long long t = threadIdx.x >= off ? part[threadIdx.x - off] : 0;
      __syncthreads();
      part[threadIdx.x] += t;
      __syncthreads();
    }
    if (M < n_mol) xoff[M] = carry + part[threadIdx.x] - cnt;
    __syncthreads();
    if (threadIdx.x == 1023) carry += part[1023];
    __syncthreads();
  }
  if (threadIdx.x == 0) xoff[n_mol] = carry;
}

// Block = one atom I (global index): [d][3n] fp32 -> scale, split, transpose.
static __global__ void __launch_bounds__(256)
prep_columns_kernel(const float* __restrict__ dense, const int64_t* __restrict__ dense_off,
                    const int32_t* __restrict__ mol_off, int n_mol, int d, const long long* __restrict__ xoff,
                    __half* __restrict__ Xh, __half* __restrict__ Xl, float* __restrict__ inv_scale) {
  __shared__ float tile[64][97];
  __shared__ float red[8];
  const int Ig = blockIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int M = owner_molecule(mol_off, n_mol, Ig);
  const int a0 = __ldg(mol_off + M), n = __ldg(mol_off + M + 1) - a0;
  const int ncol = 3 * n, npad = (ncol + 15) / 16 * 16, kKB = d / kKBlk;
  const float* src = dense + (size_t)__ldg(dense_off + M) + (size_t)(Ig - a0) * d * ncol;  // [d][ncol]
  const size_t total = (size_t)d * ncol;
  // pass 1: block absmax -> one power-of-two scale: amax * s in [2^9, 2^10)
  float amax = 0.f;
  for (size_t i = threadIdx.x; i < total; i += 256) amax = fmaxf(amax, fabsf(__ldg(src + i)));
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, m));
  if (lane == 0) red[warp] = amax;
  __syncthreads();
  amax = red[0];
#pragma unroll
  for (int w = 1; w < 8; ++w) amax = fmaxf(amax, red[w]);
  int sh = 9 - ((int)((__float_as_uint(amax) >> 23) & 0xffu) - 127);
  if (amax == 0.f) sh = 0;
  sh = sh < -100 ? -100 : (sh > 100 ? 100 : sh);
  const float s = __uint_as_float((uint32_t)(127 + sh) << 23);
  if (threadIdx.x == 0) inv_scale[Ig] = __uint_as_float((uint32_t)(127 - sh) << 23);
  // pass 2: [64 inputs][96 columns] tiles through shared memory
  const size_t row0 = (size_t)__ldg(xoff + M) + (size_t)(Ig - a0) * kKB * npad;
  for (int kb = 0; kb < kKB; ++kb) {
    for (int c0 = 0; c0 < npad; c0 += 96) {
      const int nc = npad - c0 < 96 ? npad - c0 : 96;
      __syncthreads();
      for (int rr = warp; rr < kKBlk; rr += 8)
        for (int cc = lane; cc < nc; cc += 32)
          tile[rr][cc] = (c0 + cc < ncol) ? __ldcs(src + (size_t)(kb * kKBlk + rr) * ncol + c0 + cc) * s : 0.f;
      __syncthreads();
      // one thread = one 16-byte chunk (8 inputs) of one column
      for (int item = threadIdx.x; item < nc * 8; item += 256) {
        const int cc = item >> 3, ch = item & 7;
        __half h[8], l[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          const float a = tile[ch * 8 + u][cc];
          h[u] = __float2half_rn(a);
          l[u] = __float2half_rn(a - __half2float(h[u]));
        }
        const size_t row = row0 + (size_t)kb * npad + c0 + cc;
        const size_t o = row * 64 + (size_t)((ch ^ (int)(row & 7)) << 3);
        *reinterpret_cast<uint4*>(Xh + o) = *reinterpret_cast<const uint4*>(h);
        *reinterpret_cast<uint4*>(Xl + o) = *reinterpret_cast<const uint4*>(l);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// 3. The tcgen05 kernel.
//    What bounds it: every (atom, stack) needs the atom's column tiles (hi + lo: 4 d N bytes) from L2, and one SM
//    can pull ~20 B per clock from L2 when all SMs do (measured 5.5 TB/s; multicast in clusters of 4 does not help,
//    L2 already merges up to ~4 identical requests).  The columns are therefore re-used from shared memory for kSPT
//    stacks per CTA: as many as the W tiles of kSPT stacks leave room for (d = 128: 4 stacks = 128 KB of W; d = 256:
//    1 stack = 128 KB).  Measured tensor-pipe activity: see DESIGN.md.
// ---------------------------------------------------------------------------------------------------
template <int D_>
struct MmaCfg {
  static constexpr int d = D_;
  static constexpr int kTPS = D_ / kTile;             // 128-row output tiles per stack
  static constexpr int kSPT = D_ <= 128 ? 4 : 1;      // stacks per task (CTA)
  static constexpr int kMT = kTPS * kSPT;             // output tiles (TMEM accumulators) per atom
  static constexpr int kKB = D_ / kKBlk;              // k-blocks
  static constexpr int kNMax = D_ <= 128 ? 64 : 96;   // columns per chunk (MMA N <= kNMax, multiple of 16)
  static constexpr int kStages = D_ <= 128 ? 4 : 3;   // B ring: one stage = hi + lo tile of one (atom, k-block)
  static constexpr int kTBuf = 512 / (kMT * kNMax);   // TMEM accumulator buffers (2)
  static constexpr uint32_t kABytes = kMT * kKB * kTileBytes;   // W tiles of one (element, stack group): 128 KB
  static constexpr uint32_t kStageBytes = 2 * kNMax * 128;
  static constexpr int kEpiWarps = 8;
  static constexpr int kTPW = kMT / 2;                // output tiles per epilogue warp (2 warp groups of 4 quarters)
  static constexpr int kThreads = 64 + 32 * kEpiWarps;
  static constexpr uint32_t kSmem = kABytes + kStages * kStageBytes + 512 + 1024;
  static_assert(kTBuf >= 2 && kMT % 2 == 0, "TMEM double buffering / epilogue split");
};

// Task order: molecules in groups of kMolGroup, inside a group the molecule index runs fastest, so that the CTAs that
// run at the same time read different molecules' column tiles while a molecule's tiles stay in L2 between its stacks.
constexpr int kMolGroup = 16;
__device__ __forceinline__ void task_decode(long long task, int n_mol, int n_units, int* M, int* unit) {
  const long long per_group = (long long)kMolGroup * n_units;
  const long long g = task / per_group;
  const int m0 = (int)(g * kMolGroup);
  const int gm = n_mol - m0 < kMolGroup ? n_mol - m0 : kMolGroup;   // molecules in this group
  const long long r = task - g * per_group;
  *M = m0 + (int)(r % gm);
  *unit = (int)(r / gm);
}

template <int D_>
__global__ void __launch_bounds__(MmaCfg<D_>::kThreads, 1)
sorf_rows_mma_kernel(const int32_t* __restrict__ elem, const int32_t* __restrict__ mol_off, int n_mol, int n_s,
                     int n_sg, float c, const __half* __restrict__ W16, const __half* __restrict__ Xh,
                     const __half* __restrict__ Xl, const long long* __restrict__ xoff,
                     const float* __restrict__ inv_scale, const float* __restrict__ zs, float* __restrict__ G) {
  using C = MmaCfg<D_>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint8_t* a_smem = smem;                        // [kMT][kKB] tiles of 16 KB
  uint8_t* b_smem = smem + C::kABytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(b_smem + C::kStages * C::kStageBytes);
  uint64_t* a_full = bars;                       // [kKB]   one barrier pair per k-block of the W tiles: the next
  uint64_t* a_empty = bars + C::kKB;             // [kKB]   element's tiles load k-block by k-block behind the last atom
  uint64_t* b_full = bars + 2 * C::kKB;          // [kStages]
  uint64_t* b_empty = b_full + C::kStages;       // [kStages]
  uint64_t* t_full = b_empty + C::kStages;       // [kTBuf]
  uint64_t* t_empty = t_full + C::kTBuf;         // [kTBuf]
  uint32_t* tmem_ptr_smem = reinterpret_cast<uint32_t*>(t_empty + C::kTBuf);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_grp = (n_s + C::kSPT - 1) / C::kSPT;          // stack groups per molecule
  const long long n_tasks = (long long)n_mol * n_grp;
  const int D = n_s * C::d;

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::kKB; ++i) { mbar_init(&a_full[i], 1); mbar_init(&a_empty[i], 1); }
    for (int i = 0; i < C::kStages; ++i) { mbar_init(&b_full[i], 1); mbar_init(&b_empty[i], 1); }
    for (int i = 0; i < C::kTBuf; ++i) { mbar_init(&t_full[i], 1); mbar_init(&t_empty[i], C::kEpiWarps); }
    fence_mbarrier_init();
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_ptr_smem))
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  const uint32_t tmem_base = *tmem_ptr_smem;

  if (warp == 0) {
    // ===================== producer: bulk copies of W tiles (per element run) and column tiles =====================
    if (lane == 0) {
      uint32_t n_a = 0, n_b = 0;   // element runs (W loads) / B stages issued so far
      for (long long task = blockIdx.x; task < n_tasks; task += gridDim.x) {
        int M, grp;
        task_decode(task, n_mol, n_grp, &M, &grp);
        const int s0 = grp * C::kSPT;
        const int n_st = n_s - s0 < C::kSPT ? n_s - s0 : C::kSPT;      // stacks of this task (tail group: fewer)
        const int a0 = __ldg(mol_off + M), n = __ldg(mol_off + M + 1) - a0;
        const int ncol = 3 * n, npad = (ncol + 15) / 16 * 16;
        const size_t row_m = (size_t)__ldg(xoff + M);
        for (int c0 = 0; c0 < npad; c0 += C::kNMax) {
          const int nc = npad - c0 < C::kNMax ? npad - c0 : C::kNMax;
          int e_prev = -1;
          for (int I = 0; I < n; ++I) {
            const int e = __ldg(elem + a0 + I);
            if (e != e_prev) {   // new element run: W tiles of (e, s0 .. s0 + n_st - 1), k-block by k-block
              const __half* w = W16 + ((size_t)e * n_s + s0) * (size_t)(C::kTPS * C::kKB) * (kTile * kKBlk);
#pragma unroll 1
              for (int kb = 0; kb < C::kKB; ++kb) {
                if (n_a > 0) mbar_wait(&a_empty[kb], (n_a - 1) & 1);
                mbar_expect_tx(&a_full[kb], (uint32_t)(n_st * C::kTPS) * kTileBytes);
                for (int t = 0; t < n_st * C::kTPS; ++t)   // tile t = stack t / kTPS, output tile t % kTPS
                  bulk_copy_g2s(a_smem + (t * C::kKB + kb) * kTileBytes,
                                w + (size_t)(t * C::kKB + kb) * (kTile * kKBlk), kTileBytes, &a_full[kb]);
              }
              ++n_a;
              e_prev = e;
            }
            for (int kb = 0; kb < C::kKB; ++kb, ++n_b) {
              const uint32_t st = n_b % C::kStages, use = n_b / C::kStages;
              if (use > 0) mbar_wait(&b_empty[st], (use - 1) & 1);
              const uint32_t bytes = (uint32_t)nc * 128;
              mbar_expect_tx(&b_full[st], 2 * bytes);
              const size_t row = row_m + ((size_t)I * C::kKB + kb) * npad + c0;
              uint8_t* dst = b_smem + st * C::kStageBytes;
              bulk_copy_g2s(dst, Xh + row * 64, bytes, &b_full[st]);
              bulk_copy_g2s(dst + C::kNMax * 128, Xl + row * 64, bytes, &b_full[st]);
            }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    // The MMAs are short (N <= 96: 48 clocks each), so the issue loop must cost less than that per MMA.  The WHOLE
    // warp runs the loop in lock-step and one elected lane issues: every operand of tcgen05.mma / commit then lives in
    // uniform registers (values read from memory are made provably uniform with a shuffle from lane 0).  Under
    // `if (lane == 0)` the compiler cannot know that and wraps every MMA in a vote / elect / R2UR loop of ~18
    // instructions, which capped the issue rate at one MMA per ~90 clocks.
    {
      const bool leader = elect_one_sync();
      const uint32_t tmem_base_u = __shfl_sync(0xffffffffu, tmem_base, 0);
      uint64_t a_desc[C::kMT][C::kKB], b_desc[C::kStages];
#pragma unroll
      for (int t = 0; t < C::kMT; ++t)
#pragma unroll
        for (int kb = 0; kb < C::kKB; ++kb)
          a_desc[t][kb] = make_kmajor_sw128_desc(smem_u32(a_smem + (t * C::kKB + kb) * kTileBytes));
#pragma unroll
      for (int st = 0; st < C::kStages; ++st) b_desc[st] = make_kmajor_sw128_desc(smem_u32(b_smem + st * C::kStageBytes));
      constexpr uint64_t kLoOff = (uint64_t)((C::kNMax * 128) >> 4);   // lo tile behind the hi tile, in 16-byte units
      uint32_t n_a = 0, n_b = 0, n_t = 0;
      for (long long task = blockIdx.x; task < n_tasks; task += gridDim.x) {
        int M, grp;
        task_decode(task, n_mol, n_grp, &M, &grp);
        const int s0 = grp * C::kSPT;
        const int n_tiles = (n_s - s0 < C::kSPT ? n_s - s0 : C::kSPT) * C::kTPS;
        const int a0 = __shfl_sync(0xffffffffu, __ldg(mol_off + M), 0);
        const int n = __shfl_sync(0xffffffffu, __ldg(mol_off + M + 1), 0) - a0;
        const int ncol = 3 * n, npad = (ncol + 15) / 16 * 16;
        for (int c0 = 0; c0 < npad; c0 += C::kNMax) {
          const int nc = npad - c0 < C::kNMax ? npad - c0 : C::kNMax;
          // D fp32, A/B fp16, both K-major, N = nc, M = 128
          const uint32_t idesc = (1u << 4) | ((uint32_t)(nc >> 3) << 17) | ((uint32_t)(kTile >> 4) << 24);
          int e_prev = -1;
          int e_next = __shfl_sync(0xffffffffu, __ldg(elem + a0), 0);
          for (int I = 0; I < n; ++I, ++n_t) {
            const int e = e_next;
            e_next = (I + 1 < n) ? __shfl_sync(0xffffffffu, __ldg(elem + a0 + I + 1), 0) : -1;
            const bool first_of_run = e != e_prev;
            if (first_of_run) { ++n_a; e_prev = e; }
            const bool last_of_run = e_next != e;
            const uint32_t tb = n_t % C::kTBuf, tuse = n_t / C::kTBuf;
            if (tuse > 0) mbar_wait(&t_empty[tb], (tuse - 1) & 1);
            tcgen05_fence_after();
            const uint32_t tmem_atom = tmem_base_u + tb * (C::kMT * C::kNMax);
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
                // Consecutive MMAs go to DIFFERENT accumulators (an MMA that accumulates into the tile its
                // predecessor wrote waits for it).
#pragma unroll
                for (int kk = 0; kk < kKBlk / 16; ++kk) {
                  const uint64_t adv = (uint64_t)((kk * 32) >> 4);
#pragma unroll
                  for (int t = 0; t < C::kMT; ++t)
                    if (t < n_tiles)
                      umma<true>(tmem_atom + t * C::kNMax, a_desc[t][kb] + adv, b_hi + kLoOff + adv, idesc,
                                 (kb > 0 || kk > 0) ? 1u : 0u);   // small term first
#pragma unroll
                  for (int t = 0; t < C::kMT; ++t)
                    if (t < n_tiles) umma<true>(tmem_atom + t * C::kNMax, a_desc[t][kb] + adv, b_hi + adv, idesc, 1u);
                }
                tcgen05_commit(&b_empty[st]);
                // the W tiles of this k-block may be replaced once the run's last MMAs on them have completed
                if (last_of_run) tcgen05_commit(&a_empty[kb]);
              }
              __syncwarp();
            }
            if (leader) tcgen05_commit(&t_full[tb]);
            __syncwarp();
          }
        }
      }
    }
  } else {
    // ===================== epilogue warps: thread = output feature of kTPW tiles =====================
    const int quarter = warp & 3;               // TMEM lanes [32 q, 32 q + 32) are the ones this warp may read
    const int half = (warp - 2) >> 2;           // tiles [half * kTPW, half * kTPW + kTPW)
    const int row = quarter * 32 + lane;        // output row inside a tile
    // position of feature (s, m) inside the lane-ordered sin table of the forward kernel (sorf_kernels.cuh)
    using ZS = Shape<(D_ < kMaxE ? D_ : kMaxE), (D_ < kMaxE ? 1 : D_ / kMaxE)>;
    constexpr int E = ZS::E, P = ZS::P, SPW = ZS::SPW, E4 = ZS::E4;
    const size_t zs_atom = (size_t)n_sg * E * kWarp;       // floats per atom
    uint32_t n_t = 0;
    for (long long task = blockIdx.x; task < n_tasks; task += gridDim.x) {
      int M, grp;
      task_decode(task, n_mol, n_grp, &M, &grp);
      const int s0 = grp * C::kSPT;
      const int a0 = __ldg(mol_off + M), n = __ldg(mol_off + M + 1) - a0;
      const int ncol = 3 * n, npad = (ncol + 15) / 16 * 16;
      size_t zs_idx[C::kTPW];
      bool live[C::kTPW];
      int feat[C::kTPW];
#pragma unroll
      for (int w = 0; w < C::kTPW; ++w) {
        const int t = half * C::kTPW + w;
        const int s = s0 + t / C::kTPS, m = (t % C::kTPS) * kTile + row;    // stack, output index inside the stack
        live[w] = s < n_s;
        const int sc = live[w] ? s : n_s - 1;
        const int zp = m / E, zj = m % E;
        zs_idx[w] = ((((size_t)(sc / SPW)) * E4 + zj / 4) * kWarp + (sc % SPW) * P + zp) * 4 + (zj & 3);
        feat[w] = sc * C::d + m;
      }
      for (int c0 = 0; c0 < npad; c0 += C::kNMax) {
        const int nc = npad - c0 < C::kNMax ? npad - c0 : C::kNMax;
        float acc[C::kTPW][C::kNMax];
#pragma unroll
        for (int w = 0; w < C::kTPW; ++w)
#pragma unroll
          for (int r = 0; r < C::kNMax; ++r) acc[w][r] = 0.f;
        float f_next[C::kTPW];
#pragma unroll
        for (int w = 0; w < C::kTPW; ++w)
          f_next[w] = c * __ldg(inv_scale + a0) * __ldg(zs + (size_t)a0 * zs_atom + zs_idx[w]);
        for (int I = 0; I < n; ++I, ++n_t) {
          float f[C::kTPW];
#pragma unroll
          for (int w = 0; w < C::kTPW; ++w) {
            f[w] = f_next[w];
            if (I + 1 < n)
              f_next[w] = c * __ldg(inv_scale + a0 + I + 1) * __ldg(zs + (size_t)(a0 + I + 1) * zs_atom + zs_idx[w]);
          }
          const uint32_t tb = n_t % C::kTBuf;
          mbar_wait(&t_full[tb], (n_t / C::kTBuf) & 1);
          tcgen05_fence_after();
#pragma unroll
          for (int w = 0; w < C::kTPW; ++w) {
            const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16) + tb * (C::kMT * C::kNMax) +
                                   (half * C::kTPW + w) * C::kNMax;
            if (live[w]) {
#pragma unroll
              for (int r0 = 0; r0 < C::kNMax; r0 += 32) {   // nc is a multiple of 16: pieces of 32 with a 16 tail
                if (r0 + 32 <= nc) {
                  uint32_t u[32];
                  tmem_ld_32x32b_x32(taddr + r0, u);
                  tmem_ld_wait();
#pragma unroll
                  for (int r = 0; r < 32; ++r) acc[w][r0 + r] = fmaf(f[w], __uint_as_float(u[r]), acc[w][r0 + r]);
                } else if (r0 < nc) {
                  uint32_t u[16];
                  tmem_ld_32x32b_x16(taddr + r0, u);
                  tmem_ld_wait();
#pragma unroll
                  for (int r = 0; r < 16; ++r) acc[w][r0 + r] = fmaf(f[w], __uint_as_float(u[r]), acc[w][r0 + r]);
                }
              }
            }
          }
          tcgen05_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&t_empty[tb]);
        }
#pragma unroll
        for (int w = 0; w < C::kTPW; ++w) {
          if (!live[w]) continue;
          float* dst = G + ((size_t)3 * a0 + c0) * D + feat[w];
#pragma unroll
          for (int r = 0; r < C::kNMax; ++r)
            if (r < nc && c0 + r < ncol) dst[(size_t)r * D] = acc[w][r];
        }
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
// 3b. The same kernel on CTA PAIRS (cta_group::2).  Measured with a stand-alone loop of MMAs (M 128, both operands in
//     shared memory): one MMA takes max(N / 2, 32 + N / 4) clocks -- 4 KB of A and 32 N bytes of B cross the 128 B / clock
//     shared-memory port -- whatever the number of accumulators in rotation: N = 96 costs 56 clocks for 48 clocks of
//     work, N = 64 costs 48 for 32.  In a pair every CTA reads its own 128 rows of A and only HALF of the columns of B
//     (32 + N / 8 clocks: below N / 2), and only half of every column tile has to come from L2 into each SM.
//     Mapping: the pair takes two consecutive stack groups of one molecule; CTA r keeps the W tiles of group 2 g + r
//     and runs the epilogue of its own stacks exactly as in the single-CTA kernel; the MMA of tile t has M = 256 =
//     tile t of CTA 0 on top of tile t of CTA 1.  Producers of both CTAs load their W tiles and their half of the
//     columns; the peer's MMA warp forwards its "full" barriers to the leader, the leader issues and commits to both.
// ---------------------------------------------------------------------------------------------------
template <int D_>
struct Mma2Cfg : MmaCfg<D_> {
  using B = MmaCfg<D_>;
  static constexpr int kStages2 = 2 * B::kStages;                       // half-size stages: twice as many
  static constexpr uint32_t kStageBytes2 = B::kStageBytes / 2;         // hi + lo of kNMax / 2 columns
  static constexpr uint32_t kSmem2 = B::kABytes + kStages2 * kStageBytes2 + 1024 + 1024;
};

template <int D_>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(MmaCfg<D_>::kThreads, 1)
sorf_rows_mma2_kernel(const int32_t* __restrict__ elem, const int32_t* __restrict__ mol_off, int n_mol, int n_s,
                      int n_sg, float c, const __half* __restrict__ W16, const __half* __restrict__ Xh,
                      const __half* __restrict__ Xl, const long long* __restrict__ xoff,
                      const float* __restrict__ inv_scale, const float* __restrict__ zs, float* __restrict__ G) {
  using C = Mma2Cfg<D_>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint8_t* a_smem = smem;                        // [kMT][kKB] tiles of 16 KB (this CTA's stacks)
  uint8_t* b_smem = smem + C::kABytes;           // [kStages2] x (hi, lo) of this CTA's half of the columns
  uint64_t* bars = reinterpret_cast<uint64_t*>(b_smem + C::kStages2 * C::kStageBytes2);
  uint64_t* a_full = bars;                       // [kKB]
  uint64_t* a_empty = a_full + C::kKB;           // [kKB]       (multicast commit)
  uint64_t* pa_full = a_empty + C::kKB;          // [kKB]       leader: the peer's W k-block has landed
  uint64_t* b_full = pa_full + C::kKB;           // [kStages2]
  uint64_t* b_empty = b_full + C::kStages2;      // [kStages2]  (multicast commit)
  uint64_t* pb_full = b_empty + C::kStages2;     // [kStages2]  leader: the peer's half stage has landed
  uint64_t* t_full = pb_full + C::kStages2;      // [kTBuf]     (multicast commit)
  uint64_t* t_empty = t_full + C::kTBuf;         // [kTBuf]     leader: epilogue warps of BOTH CTAs
  uint32_t* tmem_ptr_smem = reinterpret_cast<uint32_t*>(t_empty + C::kTBuf);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int n_pairs = gridDim.x >> 1, pair = blockIdx.x >> 1;
  const int n_grp = (n_s + C::kSPT - 1) / C::kSPT;          // stack groups per molecule
  const int n_gp = (n_grp + 1) / 2;                         // pairs of groups
  const long long n_tasks = (long long)n_mol * n_gp;

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::kKB; ++i) { mbar_init(&a_full[i], 1); mbar_init(&a_empty[i], 1); mbar_init(&pa_full[i], 1); }
    for (int i = 0; i < C::kStages2; ++i) { mbar_init(&b_full[i], 1); mbar_init(&b_empty[i], 1); mbar_init(&pb_full[i], 1); }
    for (int i = 0; i < C::kTBuf; ++i) { mbar_init(&t_full[i], 1); mbar_init(&t_empty[i], 2 * C::kEpiWarps); }
    fence_mbarrier_init();
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_ptr_smem))
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  tcgen05_fence_before();
  __syncthreads();
  cluster_sync_all();                              // the peer's barriers exist before anything arrives on them
  tcgen05_fence_after();
  const uint32_t tmem_base = *tmem_ptr_smem;

  // this CTA's stack group of a task (the last pair of an odd number of groups: the peer repeats the last group and
  // writes nothing)
  auto my_group = [&](int gp, bool* live_grp) {
    int g = 2 * gp + (int)rank;
    *live_grp = g < n_grp;
    return g < n_grp ? g : n_grp - 1;
  };

  if (warp == 0) {
    // ===================== producer (both CTAs): own W tiles, own half of the columns =====================
    if (lane == 0) {
      uint32_t n_a = 0, n_b = 0;
      for (long long task = pair; task < n_tasks; task += n_pairs) {
        int M, gp;
        task_decode(task, n_mol, n_gp, &M, &gp);
        bool live_grp;
        const int s0 = my_group(gp, &live_grp) * C::kSPT;
        const int n_st = n_s - s0 < C::kSPT ? n_s - s0 : C::kSPT;
        const int a0 = __ldg(mol_off + M), n = __ldg(mol_off + M + 1) - a0;
        const int ncol = 3 * n, npad = (ncol + 15) / 16 * 16;
        const size_t row_m = (size_t)__ldg(xoff + M);
        for (int c0 = 0; c0 < npad; c0 += C::kNMax) {
          const int nc = npad - c0 < C::kNMax ? npad - c0 : C::kNMax;
          const int nh = nc >> 1;                                        // this CTA's columns: [c0 + rank nh, + nh)
          int e_prev = -1;
          for (int I = 0; I < n; ++I) {
            const int e = __ldg(elem + a0 + I);
            if (e != e_prev) {
              const __half* w = W16 + ((size_t)e * n_s + s0) * (size_t)(C::kTPS * C::kKB) * (kTile * kKBlk);
#pragma unroll 1
              for (int kb = 0; kb < C::kKB; ++kb) {
                if (n_a > 0) mbar_wait(&a_empty[kb], (n_a - 1) & 1);
                mbar_expect_tx(&a_full[kb], (uint32_t)(n_st * C::kTPS) * kTileBytes);
                for (int t = 0; t < n_st * C::kTPS; ++t)
                  bulk_copy_g2s(a_smem + (t * C::kKB + kb) * kTileBytes,
                                w + (size_t)(t * C::kKB + kb) * (kTile * kKBlk), kTileBytes, &a_full[kb]);
              }
              ++n_a;
              e_prev = e;
            }
            for (int kb = 0; kb < C::kKB; ++kb, ++n_b) {
              const uint32_t st = n_b % C::kStages2, use = n_b / C::kStages2;
              if (use > 0) mbar_wait(&b_empty[st], (use - 1) & 1);
              const uint32_t bytes = (uint32_t)nh * 128;
              mbar_expect_tx(&b_full[st], 2 * bytes);
              const size_t row = row_m + ((size_t)I * C::kKB + kb) * npad + c0 + (size_t)rank * nh;
              uint8_t* dst = b_smem + st * C::kStageBytes2;
              bulk_copy_g2s(dst, Xh + row * 64, bytes, &b_full[st]);
              bulk_copy_g2s(dst + (C::kNMax / 2) * 128, Xl + row * 64, bytes, &b_full[st]);
            }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA warp: the leader issues for the pair, the peer forwards its "full" barriers ==========
    const bool leader_lane = elect_one_sync();
    const uint32_t tmem_base_u = __shfl_sync(0xffffffffu, tmem_base, 0);
    const uint32_t rank_u = __shfl_sync(0xffffffffu, rank, 0);
    uint64_t a_desc[C::kMT][C::kKB], b_desc[C::kStages2];
#pragma unroll
    for (int t = 0; t < C::kMT; ++t)
#pragma unroll
      for (int kb = 0; kb < C::kKB; ++kb)
        a_desc[t][kb] = make_kmajor_sw128_desc(smem_u32(a_smem + (t * C::kKB + kb) * kTileBytes));
#pragma unroll
    for (int st = 0; st < C::kStages2; ++st) b_desc[st] = make_kmajor_sw128_desc(smem_u32(b_smem + st * C::kStageBytes2));
    constexpr uint64_t kLoOff = (uint64_t)(((C::kNMax / 2) * 128) >> 4);
    uint32_t n_a = 0, n_b = 0, n_t = 0;
    for (long long task = pair; task < n_tasks; task += n_pairs) {
      int M, gp;
      task_decode(task, n_mol, n_gp, &M, &gp);
      // tiles of the LEADER's group (2 gp): it always has at least as many stacks as the peer's
      const int s0l = 2 * gp * C::kSPT;
      const int n_tiles = (n_s - s0l < C::kSPT ? n_s - s0l : C::kSPT) * C::kTPS;
      const int a0 = __shfl_sync(0xffffffffu, __ldg(mol_off + M), 0);
      const int n = __shfl_sync(0xffffffffu, __ldg(mol_off + M + 1), 0) - a0;
      const int ncol = 3 * n, npad = (ncol + 15) / 16 * 16;
      for (int c0 = 0; c0 < npad; c0 += C::kNMax) {
        const int nc = npad - c0 < C::kNMax ? npad - c0 : C::kNMax;
        // D fp32, A/B fp16, both K-major, N = nc (both halves), M = 256 (both CTAs)
        const uint32_t idesc = (1u << 4) | ((uint32_t)(nc >> 3) << 17) | ((uint32_t)((2 * kTile) >> 4) << 24);
        int e_prev = -1;
        int e_next = __shfl_sync(0xffffffffu, __ldg(elem + a0), 0);
        for (int I = 0; I < n; ++I, ++n_t) {
          const int e = e_next;
          e_next = (I + 1 < n) ? __shfl_sync(0xffffffffu, __ldg(elem + a0 + I + 1), 0) : -1;
          const bool first_of_run = e != e_prev;
          if (first_of_run) { ++n_a; e_prev = e; }
          const bool last_of_run = e_next != e;
          const uint32_t tb = n_t % C::kTBuf, tuse = n_t / C::kTBuf;
          if (rank_u == 0) {
            if (tuse > 0) mbar_wait(&t_empty[tb], (tuse - 1) & 1);
            tcgen05_fence_after();
          }
          const uint32_t tmem_atom = tmem_base_u + tb * (C::kMT * C::kNMax);
#pragma unroll
          for (int kb = 0; kb < C::kKB; ++kb, ++n_b) {
            const uint32_t st = n_b % C::kStages2;
            if (first_of_run) mbar_wait(&a_full[kb], (n_a - 1) & 1);
            mbar_wait(&b_full[st], (n_b / C::kStages2) & 1);
            if (rank_u != 0) {
              // peer: this k-block of W and this half stage are in my shared memory -- tell the leader
              if (leader_lane) {
                if (first_of_run) mbar_arrive_remote(&pa_full[kb], 0);
                mbar_arrive_remote(&pb_full[st], 0);
              }
              __syncwarp();
              continue;
            }
            if (first_of_run) mbar_wait(&pa_full[kb], (n_a - 1) & 1);
            mbar_wait(&pb_full[st], (n_b / C::kStages2) & 1);
            tcgen05_fence_after();
            uint64_t b_hi = b_desc[0];
#pragma unroll
            for (int q = 1; q < C::kStages2; ++q) b_hi = (st == (uint32_t)q) ? b_desc[q] : b_hi;
            if (leader_lane) {
#pragma unroll
              for (int kk = 0; kk < kKBlk / 16; ++kk) {
                const uint64_t adv = (uint64_t)((kk * 32) >> 4);
#pragma unroll
                for (int t = 0; t < C::kMT; ++t)
                  if (t < n_tiles)
                    umma2<true>(tmem_atom + t * C::kNMax, a_desc[t][kb] + adv, b_hi + kLoOff + adv, idesc,
                                (kb > 0 || kk > 0) ? 1u : 0u);   // small term first
#pragma unroll
                for (int t = 0; t < C::kMT; ++t)
                  if (t < n_tiles) umma2<true>(tmem_atom + t * C::kNMax, a_desc[t][kb] + adv, b_hi + adv, idesc, 1u);
              }
              tcgen05_commit2(&b_empty[st]);                      // both producers may refill this stage
              if (last_of_run) tcgen05_commit2(&a_empty[kb]);     // both producers may replace this k-block of W
            }
            __syncwarp();
          }
          if (rank_u == 0 && leader_lane) tcgen05_commit2(&t_full[tb]);   // accumulators of both CTAs complete
          __syncwarp();
        }
      }
    }
  } else {
    // ===================== epilogue warps (both CTAs): thread = output feature of this CTA's stacks =====================
    const int quarter = warp & 3;
    const int half = (warp - 2) >> 2;
    const int row = quarter * 32 + lane;
    using ZS = Shape<(D_ < kMaxE ? D_ : kMaxE), (D_ < kMaxE ? 1 : D_ / kMaxE)>;
    constexpr int E = ZS::E, P = ZS::P, SPW = ZS::SPW, E4 = ZS::E4;
    const size_t zs_atom = (size_t)n_sg * E * kWarp;
    uint32_t n_t = 0;
    for (long long task = pair; task < n_tasks; task += n_pairs) {
      int M, gp;
      task_decode(task, n_mol, n_gp, &M, &gp);
      bool live_grp;
      const int s0 = my_group(gp, &live_grp) * C::kSPT;
      const int a0 = __ldg(mol_off + M), n = __ldg(mol_off + M + 1) - a0;
      const int ncol = 3 * n, npad = (ncol + 15) / 16 * 16;
      size_t zs_idx[C::kTPW];
      bool live[C::kTPW];
      int feat[C::kTPW];
#pragma unroll
      for (int w = 0; w < C::kTPW; ++w) {
        const int t = half * C::kTPW + w;
        const int s = s0 + t / C::kTPS, m = (t % C::kTPS) * kTile + row;
        live[w] = live_grp && s < n_s;
        const int sc = s < n_s ? s : n_s - 1;
        const int zp = m / E, zj = m % E;
        zs_idx[w] = ((((size_t)(sc / SPW)) * E4 + zj / 4) * kWarp + (sc % SPW) * P + zp) * 4 + (zj & 3);
        feat[w] = sc * C::d + m;
      }
      for (int c0 = 0; c0 < npad; c0 += C::kNMax) {
        const int nc = npad - c0 < C::kNMax ? npad - c0 : C::kNMax;
        float acc[C::kTPW][C::kNMax];
#pragma unroll
        for (int w = 0; w < C::kTPW; ++w)
#pragma unroll
          for (int r = 0; r < C::kNMax; ++r) acc[w][r] = 0.f;
        float f_next[C::kTPW];
#pragma unroll
        for (int w = 0; w < C::kTPW; ++w)
          f_next[w] = c * __ldg(inv_scale + a0) * __ldg(zs + (size_t)a0 * zs_atom + zs_idx[w]);
        for (int I = 0; I < n; ++I, ++n_t) {
          float f[C::kTPW];
#pragma unroll
          for (int w = 0; w < C::kTPW; ++w) {
            f[w] = f_next[w];
            if (I + 1 < n)
              f_next[w] = c * __ldg(inv_scale + a0 + I + 1) * __ldg(zs + (size_t)(a0 + I + 1) * zs_atom + zs_idx[w]);
          }
          const uint32_t tb = n_t % C::kTBuf;
          mbar_wait(&t_full[tb], (n_t / C::kTBuf) & 1);
          tcgen05_fence_after();
#pragma unroll
          for (int w = 0; w < C::kTPW; ++w) {
            const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16) + tb * (C::kMT * C::kNMax) +
                                   (half * C::kTPW + w) * C::kNMax;
            if (live[w]) {
#pragma unroll
              for (int r0 = 0; r0 < C::kNMax; r0 += 32) {
                if (r0 + 32 <= nc) {
                  uint32_t u[32];
                  tmem_ld_32x32b_x32(taddr + r0, u);
                  tmem_ld_wait();
#pragma unroll
                  for (int r = 0; r < 32; ++r) acc[w][r0 + r] = fmaf(f[w], __uint_as_float(u[r]), acc[w][r0 + r]);
                } else if (r0 < nc) {
                  uint32_t u[16];
                  tmem_ld_32x32b_x16(taddr + r0, u);
                  tmem_ld_wait();
#pragma unroll
                  for (int r = 0; r < 16; ++r) acc[w][r0 + r] = fmaf(f[w], __uint_as_float(u[r]), acc[w][r0 + r]);
                }
              }
            }
          }
          tcgen05_fence_before();
          __syncwarp();
          if (lane == 0) {                       // the leader's MMA warp waits for the epilogues of both CTAs
            if (rank == 0) mbar_arrive(&t_empty[tb]); else mbar_arrive_remote(&t_empty[tb], 0);
          }
        }
#pragma unroll
        for (int w = 0; w < C::kTPW; ++w) {
          if (!live[w]) continue;
          float* dst = G + ((size_t)3 * a0 + c0) * (size_t)(n_s * C::d) + feat[w];
#pragma unroll
          for (int r = 0; r < C::kNMax; ++r)
            if (r < nc && c0 + r < ncol) dst[(size_t)r * (n_s * C::d)] = acc[w][r];
        }
      }
    }
  }

  tcgen05_fence_before();
  __syncthreads();
  cluster_sync_all();                              // nobody leaves while the peer may still touch its memory
  if (warp == 2) {
    tcgen05_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
  }
}

// ---------------------------------------------------------------------------------------------------
// Host side
// ---------------------------------------------------------------------------------------------------
int sorf_mma_build_w(const qmll_sorf_params* p, const SorfTables& t, void* W16, cudaStream_t st) {
  const int n_s = p->D / p->d;
  if (p->d == 128) {
    using S = Shape<shape_E(128), shape_P(128)>;
    const int n_sg = (n_s + S::SPW - 1) / S::SPW;
    const long long w_tasks = (long long)p->n_elem * n_sg * p->d;
    build_w_kernel<S><<<(unsigned)((w_tasks + 3) / 4), kFwdThreads, 0, st>>>(t.sign_bits, p->n_elem, n_s, n_sg,
                                                                            p->n_transform, (__half*)W16);
  } else if (p->d == 256) {
    using S = Shape<shape_E(256), shape_P(256)>;
    const int n_sg = (n_s + S::SPW - 1) / S::SPW;
    const long long w_tasks = (long long)p->n_elem * n_sg * p->d;
    build_w_kernel<S><<<(unsigned)((w_tasks + 3) / 4), kFwdThreads, 0, st>>>(t.sign_bits, p->n_elem, n_s, n_sg,
                                                                            p->n_transform, (__half*)W16);
  } else {
    return QMLL_ERR_UNSUPPORTED;
  }
  QMLL_LAUNCH_CHECK("build_w_kernel");
  return QMLL_OK;
}

bool sorf_mma_supported(const qmll_sorf_params* p) {
  return (p->d == 128 || p->d == 256) && p->n_transform >= 1 && p->n_transform <= 3;
}

// bytes of the W table, of ONE of the two column arrays (upper bound: n * kKB * roundup16(3n) rows of 128 bytes per
// molecule <= 2 * (dense_floats + 15 d n_atoms) bytes) and of the per-molecule offsets / per-atom scales
size_t sorf_mma_w_bytes(const qmll_sorf_params* p) { return (size_t)p->n_elem * (p->D / p->d) * p->d * p->d * sizeof(__half); }
size_t sorf_mma_x_bytes(const qmll_sorf_params* p, int64_t n_atoms, int64_t dense_floats) {
  return (size_t)2 * ((size_t)dense_floats + (size_t)15 * p->d * (size_t)n_atoms) + 1024;
}

template <int D_>
static int launch_rows_mma(const SorfProblem& pr, const SorfTables& t, const float* zs, const qmll_grad* grad,
                           __half* W16, __half* Xh, __half* Xl, long long* xoff, float* inv_scale, float* G,
                           cudaStream_t st, bool pairs) {
  using S = Shape<shape_E(D_), shape_P(D_)>;
  using C = MmaCfg<D_>;
  const qmll_sorf_params* p = pr.p;
  const int n_s = p->D / p->d, n_sg = (n_s + S::SPW - 1) / S::SPW;
  const long long w_tasks = (long long)p->n_elem * n_sg * p->d;
  build_w_kernel<S><<<(unsigned)((w_tasks + 3) / 4), kFwdThreads, 0, st>>>(t.sign_bits, p->n_elem, n_s, n_sg,
                                                                          p->n_transform, W16);
  QMLL_LAUNCH_CHECK("build_w_kernel");
  x_offsets_kernel<<<1, 1024, 0, st>>>(pr.mol_off, pr.n_mol, C::kKB, xoff);
  QMLL_LAUNCH_CHECK("x_offsets_kernel");
  prep_columns_kernel<<<(unsigned)pr.n_atoms, 256, 0, st>>>(grad->dense, grad->dense_off, pr.mol_off, pr.n_mol, p->d,
                                                           xoff, Xh, Xl, inv_scale);
  QMLL_LAUNCH_CHECK("prep_columns_kernel");
  const float c = (float)(sqrt((double)p->d) / (double)p->sigma * pow((double)p->d, -0.5 * p->n_transform));
  const int n_grp = (n_s + C::kSPT - 1) / C::kSPT;
  if (pairs) {
    using C2 = Mma2Cfg<D_>;
    auto kern = sorf_rows_mma2_kernel<D_>;
    QMLL_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C2::kSmem2));
    const long long n_tasks = (long long)pr.n_mol * ((n_grp + 1) / 2);
    const int max_pairs = device_sm_count() / 2;
    const int n_pairs = (int)(n_tasks < max_pairs ? n_tasks : max_pairs);
    kern<<<2 * n_pairs, C::kThreads, C2::kSmem2, st>>>(pr.elem, pr.mol_off, pr.n_mol, n_s, n_sg, c, W16, Xh, Xl, xoff,
                                                       inv_scale, zs, G);
    QMLL_LAUNCH_CHECK("sorf_rows_mma2_kernel");
    return QMLL_OK;
  }
  auto kern = sorf_rows_mma_kernel<D_>;
  QMLL_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::kSmem));
  const long long n_tasks = (long long)pr.n_mol * n_grp;
  const int grid = (int)(n_tasks < device_sm_count() ? n_tasks : device_sm_count());
  kern<<<grid, C::kThreads, C::kSmem, st>>>(pr.elem, pr.mol_off, pr.n_mol, n_s, n_sg, c, W16, Xh, Xl, xoff,
                                            inv_scale, zs, G);
  QMLL_LAUNCH_CHECK("sorf_rows_mma_kernel");
  return QMLL_OK;
}

int sorf_force_rows_dense_mma(const SorfProblem& pr, const SorfTables& t, const float* zs, const qmll_grad* grad,
                              void* W16, void* Xh, void* Xl, long long* xoff, float* inv_scale, float* G,
                              cudaStream_t st, bool pairs) {
  if (pr.n_atoms == 0 || pr.n_mol == 0) return QMLL_OK;
  if (pr.p->d == 128)
    return launch_rows_mma<128>(pr, t, zs, grad, (__half*)W16, (__half*)Xh, (__half*)Xl, xoff, inv_scale, G, st, pairs);
  if (pr.p->d == 256)
    return launch_rows_mma<256>(pr, t, zs, grad, (__half*)W16, (__half*)Xh, (__half*)Xl, xoff, inv_scale, G, st, pairs);
  return QMLL_ERR_UNSUPPORTED;
}

}  // namespace qmll
