// solve_kernels.cu -- NEXT #1 of SURVEY.md section 8(f): alpha = (ZtZ + lambda I)^-1 Zty  (eq. 16-17;
// "solved by LU decomposition", L137 -- the matrix is symmetric positive definite, so Cholesky).  FP64 throughout: the
// Gram matrix of random features is ill-conditioned (the paper's FP32 round-off remark, L351), and the O(D^3/3) solve
// is small beside the O(rows D^2) accumulation.  Two-level blocked right-looking Cholesky:
//   potrf_diag_kernel (64 x 64 diagonal block, one row per thread in registers)  ->  trsm_panel_kernel (thread per
//   row, column-oriented substitution)  ->  syrk_update_kernel on the 256-wide panel's own columns; after the panel
//   one rank-256 syrk_update_kernel of the trailing matrix,
// the right-hand side rides along as row D of the working matrix (so L y = b costs nothing extra), then the backward
// substitution in one kernel whose CTAs hand the solved blocks to one another through flags (trsv_back_kernel).
// syrk_update_kernel is the O(D^3) part: 128 x 64 tiles on the FP64 tensor-core path (mma.sync.m8n8k4.f64, DMMA: the
// measured peak, profiles/peaks_r2.json kinds 13 / 14, is 18.5 T FMA/s against 17.0 for scalar DFMA, with 1/8 of the
// instructions and 1/5 of the shared-memory loads), operands through a 2-stage cp.async ring, three CTAs per SM (the
// third fills the issue gaps between a warp's dependent DMMAs: pipe 82 % -> 90 % busy).
// `info` (device int) follows LAPACK: 0 = success, k > 0 = the leading minor of order k is not positive definite (the
// factorisation then carries NaNs).  The working matrix has leading dimension ld = D rounded up to 8 (16-byte copies).
#include <mutex>

#include "qmll_common.cuh"

namespace qmll {

constexpr int kNB = 64;     // inner step: diagonal block factorised in registers
constexpr int kNB2 = 256;   // outer panel: one trailing update per 256 columns

static inline int solve_ld(int D) { return (D + 7) & ~7; }

// The 64 x 64 diagonal block goes to shared memory by 8-byte cp.async: all of a thread's copies are in flight at once
// (a load -> store loop serialised one L2 round trip per unrolled group and was half of every panel kernel's time).
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// M = lower triangle of ZtZ + lambda I in FP64 (row i, columns 0 .. i; the upper triangle is never read), row D = Zty
__global__ void __launch_bounds__(256) solve_prepare_kernel(const float* __restrict__ ZtZ, const float* __restrict__ Zty,
                                                            int D, int ld, double lambda, double* __restrict__ M,
                                                            double* __restrict__ rhs, int* __restrict__ info,
                                                            int* __restrict__ flags, int n_flags) {
  const int i = blockIdx.y;
  const int j = blockIdx.x * 1024 + threadIdx.x * 4;
  if (blockIdx.x == 0 && i == 0) {
    if (threadIdx.x == 0) *info = 0;
    for (int k = threadIdx.x; k < n_flags; k += 256) flags[k] = 0;
  }
  if (i == D) {
#pragma unroll
    for (int q = 0; q < 4; ++q)
      if (j + q < D) rhs[j + q] = (double)Zty[j + q];
    return;
  }
  if (j > i) return;
  const float* src = ZtZ + (size_t)i * D + j;
  double* dst = M + (size_t)i * ld + j;
#pragma unroll
  for (int q = 0; q < 4; ++q)
    if (j + q <= i) dst[q] = (double)src[q] + (j + q == i ? lambda : 0.0);
}

// Cholesky of the nb x nb diagonal block at (k0, k0): A = L L^T, L overwrites the lower triangle.  The block lives in
// shared memory and is factorised in four block columns of 16 (right-looking between them):
//   * panel: threads 0..63 = rows, the row's 16 entries in registers; per column ONE 64-thread named barrier -- every
//     thread publishes its entry of column j, reads the pivot and the column back, and updates the (at most 15)
//     remaining entries of its row: the serial chain per column is barrier + rsqrt + two multiplies + one FMA;
//   * update: all 256 threads subtract the rank-16 product from the rest of the block (items of 1 row x 4 columns).
// History: a register-resident 64-wide row with 63 FMAs per column and thread (rolled by shifting the row one
// register per column; fully unrolled it was 93 KB of straight-line code at instruction-fetch speed) took 22 us: one
// warp per scheduler issues its ~200 instructions per column in order, behind the chain.
// Rows / columns >= nb are an identity pad.
constexpr int kPB = 16;
__global__ void __launch_bounds__(256) potrf_diag_kernel(double* __restrict__ M, int ld, int k0, int nb, int* info) {
  __shared__ double tile[kNB][kNB + 1];
  __shared__ double col[2][kNB];
  const int t = threadIdx.x;
  for (int idx = t; idx < kNB * kNB; idx += 256) {
    const int r = idx / kNB, c = idx % kNB;
    if (r < nb && c <= r) cp_async8(&tile[r][c], M + (size_t)(k0 + r) * ld + k0 + c);
    else tile[r][c] = r == c ? 1.0 : 0.0;
  }
  cp_async_wait_all();
  __syncthreads();
#pragma unroll 1
  for (int c0 = 0; c0 < kNB; c0 += kPB) {
    if (t < kNB) {                                       // ---- panel: rows 0..63 (rows above c0 carry zeros along)
      const int i = t;
      double a[kPB];
#pragma unroll
      for (int q = 0; q < kPB; ++q) a[q] = i >= c0 ? tile[i][c0 + q] : 0.0;
#pragma unroll
      for (int q = 0; q < kPB; ++q) {
        const int j = c0 + q;
        col[q & 1][i] = a[q];
        asm volatile("bar.sync 1, 64;" ::: "memory");
        const double piv = col[q & 1][j];
        if (i == j && j < nb && !(piv > 0.0) && *info == 0) *info = k0 + j + 1;
        const double dinv = rsqrt(piv);
        a[q] *= dinv;                                     // row j: sqrt(piv); rows below: l_ij; rows above: 0
        const double sc = a[q] * dinv;                    // l_ij / sqrt(piv); col[c] * (1 / sqrt(piv)) = l_cj
#pragma unroll
        for (int k = q + 1; k < kPB; ++k) a[k] = fma(-sc, col[q & 1][c0 + k], a[k]);
      }
      if (i >= c0) {
#pragma unroll
        for (int q = 0; q < kPB; ++q)
          if (c0 + q <= i) tile[i][c0 + q] = a[q];
      }
    }
    __syncthreads();
    // ---- rank-16 update of rows / columns >= c0 + 16 (lower triangle): item = (row, 4 columns)
    const int r0 = c0 + kPB, R = kNB - r0;
    for (int idx = t; idx < R * (R / 4); idx += 256) {
      const int i = r0 + idx % R, cb = r0 + 4 * (idx / R);
      if (cb > i) continue;
      double li[kPB], s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
      for (int k = 0; k < kPB; ++k) li[k] = tile[i][c0 + k];
#pragma unroll
      for (int k = 0; k < kPB; ++k) {
        s0 = fma(li[k], tile[cb][c0 + k], s0);
        s1 = fma(li[k], tile[cb + 1][c0 + k], s1);
        s2 = fma(li[k], tile[cb + 2][c0 + k], s2);
        s3 = fma(li[k], tile[cb + 3][c0 + k], s3);
      }
      tile[i][cb] -= s0;                                  // entries above the diagonal are scratch (never read back)
      tile[i][cb + 1] -= s1;
      tile[i][cb + 2] -= s2;
      tile[i][cb + 3] -= s3;
    }
    __syncthreads();
  }
  for (int idx = t; idx < nb * nb; idx += 256) {
    const int r = idx / nb, c = idx % nb;
    if (c <= r) M[(size_t)(k0 + r) * ld + k0 + c] = tile[r][c];
  }
}

// Rows below the nb x nb diagonal block (rows k0 + nb .. n_rows - 1): X = A21 L11^-T, one thread per row,
// column-oriented forward substitution (x_c final -> every later x_k gets its term: independent FMAs); L11 transposed
// in shared memory so that one broadcast LDS.128 serves two FMAs.  Columns >= nb are an identity pad.
constexpr int kLtLd = kNB + 2;
__global__ void __launch_bounds__(128) trsm_panel_kernel(double* __restrict__ M, int n_rows, int ld, int k0, int nb) {
  __shared__ __align__(16) double lt[kNB][kLtLd];   // lt[c][k] = L11[k][c]
  __shared__ double dinv[kNB];
  for (int idx = threadIdx.x; idx < kNB * kNB; idx += 128) {
    const int r = idx / kNB, c = idx % kNB;
    if (r < nb && c < nb) cp_async8(&lt[c][r], M + (size_t)(k0 + r) * ld + k0 + c);
    else lt[c][r] = r == c ? 1.0 : 0.0;
  }
  cp_async_wait_all();
  __syncthreads();
  if (threadIdx.x < kNB) dinv[threadIdx.x] = 1.0 / lt[threadIdx.x][threadIdx.x];
  __syncthreads();
  const int i = k0 + nb + blockIdx.x * 128 + threadIdx.x;
  if (i >= n_rows) return;
  double2* row = reinterpret_cast<double2*>(M + (size_t)i * ld + k0);
  double x[kNB];
  if (nb == kNB) {
#pragma unroll
    for (int c = 0; c < kNB; c += 2) { const double2 v = row[c / 2]; x[c] = v.x; x[c + 1] = v.y; }
  } else {
#pragma unroll
    for (int c = 0; c < kNB; ++c) x[c] = c < nb ? M[(size_t)i * ld + k0 + c] : 0.0;
  }
#pragma unroll
  for (int c = 0; c < kNB; ++c) {
    x[c] *= dinv[c];
    const double xc = x[c];
    int k = c + 1;
    if (k & 1) { if (k < kNB) x[k] = fma(-xc, lt[c][k], x[k]); ++k; }
#pragma unroll
    for (; k < kNB; k += 2) {
      const double2 l2 = *reinterpret_cast<const double2*>(&lt[c][k]);
      x[k] = fma(-xc, l2.x, x[k]);
      x[k + 1] = fma(-xc, l2.y, x[k + 1]);
    }
  }
  if (nb == kNB) {
#pragma unroll
    for (int c = 0; c < kNB; c += 2) row[c / 2] = make_double2(x[c], x[c + 1]);
  } else {
#pragma unroll
    for (int c = 0; c < kNB; ++c)
      if (c < nb) M[(size_t)i * ld + k0 + c] = x[c];
  }
}

// Symmetric rank-kn update on the lower triangle:  C[i][j] -= sum_{m < kn} M[i][k0 + m] * M[j][k0 + m]  for rows
// i >= r0, columns c0 <= j < c1, j <= i (c0 even).  CTA = 128 x 64 tile (blockIdx.x: row tile from r0, blockIdx.y:
// column tile from c0), 4 warps as 2 x 2, warp tile 64 x 32 = 8 x 4 DMMA tiles (128 accumulator registers).  Both
// operands are row-major slices of M with k contiguous, which is exactly the m8n8k4 fragment order (A: row lane / 4,
// k lane % 4; B the same with the row as n), so the stages are plain copies: [rows][16 k] with a row pitch of 20
// doubles (conflict-free LDS.64 for the 8 rows x 4 k a fragment touches), filled by 16-byte cp.async (zero-filled
// beyond kn and beyond the last row).  n_rows = D + 1: the extra row carries the right-hand side.
constexpr int kUM = 128, kUN = 64, kUK = 16, kUPitch = 20, kUStages = 2;
constexpr int kUStageDoubles = (kUM + kUN) * kUPitch;
constexpr int kUSmemBytes = kUStages * kUStageDoubles * 8;

__device__ __forceinline__ void cp_async16_zfill(uint32_t dst, const void* src, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void dmma_m8n8k4(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(128, 3) syrk_update_kernel(double* __restrict__ M, int n_rows, int ld, int r0, int c0,
                                                             int c1, int k0, int kn) {
  const int i0 = r0 + blockIdx.x * kUM, j0 = c0 + blockIdx.y * kUN;
  if (j0 >= c1 || j0 > i0 + kUM - 1) return;          // tile entirely above the diagonal or outside the column range
  extern __shared__ __align__(16) double usm[];
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const int wr = warp >> 1, wc = warp & 1, g = lane >> 2, tg = lane & 3;
  const uint32_t usm_addr = (uint32_t)__cvta_generic_to_shared(usm);

  // loader: a stage is 192 rows x 8 pieces of 16 bytes; thread t copies piece t % 8 of rows t / 8 + 16 q, q < 12
  const int lrow = t >> 3, lch = t & 7;
  auto load_stage = [&](int chunk, int slot) {
    const int kk = chunk * kUK + lch * 2;
    int bytes = (kn - kk) * 8;
    bytes = bytes < 0 ? 0 : (bytes > 16 ? 16 : bytes);
    const double* col = M + k0 + (bytes ? kk : 0);
    const uint32_t dst = usm_addr + (uint32_t)((slot * kUStageDoubles + lrow * kUPitch + lch * 2) * 8);
#pragma unroll
    for (int q = 0; q < 12; ++q) {
      const int gr = q < 8 ? i0 + lrow + 16 * q : j0 + lrow + 16 * (q - 8);
      const bool ok = gr < n_rows;
      cp_async16_zfill(dst + (uint32_t)(16 * q * kUPitch * 8), col + (size_t)(ok ? gr : 0) * ld, ok ? bytes : 0);
    }
  };

  double acc[8][4][2];
#pragma unroll
  for (int u = 0; u < 8; ++u)
#pragma unroll
    for (int v = 0; v < 4; ++v) acc[u][v][0] = acc[u][v][1] = 0.0;

  const int n_chunks = (kn + kUK - 1) / kUK;
#pragma unroll
  for (int s = 0; s < kUStages - 1; ++s) {
    if (s < n_chunks) load_stage(s, s);
    asm volatile("cp.async.commit_group;" ::: "memory");
  }
  for (int ch = 0; ch < n_chunks; ++ch) {
    asm volatile("cp.async.wait_group %0;" ::"n"(kUStages - 2) : "memory");
    __syncthreads();                    // stage ch has landed for every thread; slot (ch - 1) % stages is free again
    if (ch + kUStages - 1 < n_chunks) load_stage(ch + kUStages - 1, (ch + kUStages - 1) % kUStages);
    asm volatile("cp.async.commit_group;" ::: "memory");
    const double* A = usm + (ch % kUStages) * kUStageDoubles + (wr * 64 + g) * kUPitch + tg;
    const double* B = usm + (ch % kUStages) * kUStageDoubles + (kUM + wc * 32 + g) * kUPitch + tg;
#pragma unroll
    for (int k4 = 0; k4 < kUK / 4; ++k4) {
      double a[8], b[4];
#pragma unroll
      for (int u = 0; u < 8; ++u) a[u] = A[u * 8 * kUPitch + k4 * 4];
#pragma unroll
      for (int v = 0; v < 4; ++v) b[v] = B[v * 8 * kUPitch + k4 * 4];
#pragma unroll
      for (int u = 0; u < 8; ++u)
#pragma unroll
        for (int v = 0; v < 4; ++v) dmma_m8n8k4(acc[u][v][0], acc[u][v][1], a[u], b[v]);
    }
  }
  // epilogue: the thread holds C[row g][columns 2 tg, 2 tg + 1] of every 8 x 8 tile
#pragma unroll
  for (int u = 0; u < 8; ++u) {
    const int i = i0 + wr * 64 + 8 * u + g;
    if (i >= n_rows) continue;
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      const int j = j0 + wc * 32 + 8 * v + 2 * tg;
      double* p = M + (size_t)i * ld + j;
      // fire-and-forget reductions (RED.ADD.F64): every element belongs to exactly one thread of one CTA, so the
      // result is deterministic, and no load latency is exposed at the end of the tile (a read-modify-write epilogue
      // cost 30 % of the warp stalls)
      if (j <= i && j < c1) atomicAdd(p, -acc[u][v][0]);
      if (j + 1 <= i && j + 1 < c1) atomicAdd(p + 1, -acc[u][v][1]);
    }
  }
}

// Backward substitution L^T a = y in ONE kernel (the forward substitution L y = b needs none: the right-hand side
// rides through the factorisation as row D of the working matrix, so that trsm_panel_kernel solves it and
// syrk_update_kernel updates it like any other row).  CTA b owns the 128 entries j in [128 b, 128 b + 128) -- thread =
// entry, the running value lives in a register -- and walks the 64-wide blocks kb from the last one down to its own:
//   * the owner of block kb (b = kb / 2) solves the diagonal block with L11^T (warp 0: two rows per lane, the solved
//     entry travels by shuffle), writes sol[k0 .. k0 + nb) and raises flag[kb] (release);
//   * every CTA below waits for the flag (acquire), then subtracts sum_m L[k0 + m][j] sol[k0 + m] from its entries;
//     its 64 values of L are loaded BEFORE the wait.
// A CTA depends only on CTAs with larger b; b is handed out by an atomic ticket in reverse, so whatever a CTA waits
// for belongs to a CTA that has already started: no co-residency requirement, no deadlock.  256 launches of 16 us
// (4.2 ms at D = 16384) became one kernel.
__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_gpu(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

constexpr int kTrsvSmemBytes = (2 * kNB * (kNB + 1) + 2 * kNB) * 8;
__global__ void __launch_bounds__(128) trsv_back_kernel(const double* __restrict__ M, int D, int ld,
                                                        const double* __restrict__ y, double* __restrict__ sol,
                                                        int* __restrict__ flags, int* __restrict__ ticket) {
  extern __shared__ __align__(16) double tsm[];           // the two diagonal blocks this CTA owns + their 1 / l_cc
  double (*tiles)[kNB][kNB + 1] = reinterpret_cast<double (*)[kNB][kNB + 1]>(tsm);
  double (*dinv2)[kNB] = reinterpret_cast<double (*)[kNB]>(tsm + 2 * kNB * (kNB + 1));
  __shared__ double s_sol[kNB];
  __shared__ double s_run[2 * kNB];
  __shared__ int s_b;
  const int t = threadIdx.x, lane = t & 31;
  if (t == 0) s_b = (int)gridDim.x - 1 - atomicAdd(ticket, 1);
  __syncthreads();
  const int b = s_b;
  const int j = b * 128 + t;
  double r = j < D ? y[j] : 0.0;
  const int n_blk = (D + kNB - 1) / kNB;
  // both owned diagonal blocks are fetched now: by the time their turn comes (after every later block) they are here,
  // and the load is off the chain of dependent block solves
  for (int o = 0; o < 2; ++o) {
    const int kb = 2 * b + o, k0 = kb * kNB, nb = kb < n_blk ? (D - k0 < kNB ? D - k0 : kNB) : 0;
    for (int idx = t; idx < kNB * kNB; idx += 128) {
      const int rr = idx / kNB, c = idx % kNB;
      if (rr < nb && c <= rr) cp_async8(&tiles[o][rr][c], M + (size_t)(k0 + rr) * ld + k0 + c);
      else tiles[o][rr][c] = rr == c ? 1.0 : 0.0;
    }
  }
  cp_async_wait_all();
  __syncthreads();
  dinv2[t >> 6][t & 63] = 1.0 / tiles[t >> 6][t & 63][t & 63];
  __syncthreads();
  for (int kb = n_blk - 1; kb >= 2 * b; --kb) {
    const int k0 = kb * kNB, nb = D - k0 < kNB ? D - k0 : kNB;
    const bool upd = j < k0;                              // this entry receives block kb's term
    double lc[kNB];                                       // L[k0 + m][j]: issued before the wait
#pragma unroll
    for (int m = 0; m < kNB; ++m) lc[m] = (upd && m < nb) ? M[(size_t)(k0 + m) * ld + j] : 0.0;
    if ((kb >> 1) == b) {                                 // owner: diagonal solve
      const double (*l)[kNB + 1] = tiles[kb & 1];
      const double* dinv = dinv2[kb & 1];
      s_run[t] = r;
      __syncthreads();
      if (t < 32) {
        const int o = (kb & 1) * kNB;                     // the block's entries sit in threads o .. o + 63
        double b0 = lane < nb ? s_run[o + lane] : 0.0, b1 = lane + 32 < nb ? s_run[o + 32 + lane] : 0.0;
        for (int c = kNB - 1; c >= 0; --c) {
          const double bc = __shfl_sync(0xffffffffu, c < 32 ? b0 : b1, c & 31) * dinv[c];
          if (lane == (c & 31)) { if (c < 32) b0 = bc; else b1 = bc; }
          if (lane < c) b0 = fma(-l[c][lane], bc, b0);
          if (lane + 32 < c) b1 = fma(-l[c][lane + 32], bc, b1);
        }
        s_sol[lane] = b0; s_sol[lane + 32] = b1;
        if (lane < nb) sol[k0 + lane] = b0;
        if (lane + 32 < nb) sol[k0 + 32 + lane] = b1;
      }
      __syncthreads();
      if (t == 0) { __threadfence(); st_release_gpu(flags + kb, 1); }
    } else {
      if (t == 0) while (ld_acquire_gpu(flags + kb) == 0) {}
      __syncthreads();
      if (t < kNB) s_sol[t] = t < nb ? __ldcg(sol + k0 + t) : 0.0;
      __syncthreads();
    }
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
    for (int m = 0; m < kNB; m += 4) {
      s0 = fma(lc[m], s_sol[m], s0);
      s1 = fma(lc[m + 1], s_sol[m + 1], s1);
      s2 = fma(lc[m + 2], s_sol[m + 2], s2);
      s3 = fma(lc[m + 3], s_sol[m + 3], s3);
    }
    r -= (s0 + s1) + (s2 + s3);
    __syncthreads();                                      // s_sol / s_run are rewritten in the next round
  }
}

__global__ void solve_finish_kernel(const double* __restrict__ sol, float* __restrict__ alpha, int D) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < D) alpha[i] = (float)sol[i];
}

// working matrix: D + 1 rows (row D = right-hand side) plus one row of slack for 16-byte accesses at the end
size_t solve_workspace_bytes(int32_t D) {
  return align_up((size_t)(D + 2) * solve_ld(D) * 8, 256) + align_up((size_t)D * 8, 256) +
         align_up((size_t)((D + kNB - 1) / kNB + 1) * 4, 256) + 512;
}

// Look-ahead (the classic one): the panel steps are short, serial kernels that leave the GPU mostly idle, so panel
// P + 1 is factorised on an internal high-priority stream WHILE the caller's stream runs the rank-256 update of the
// rest of the trailing matrix with panel P.  Per panel: [hi] factor P, update only the columns of panel P + 1 ->
// [caller] update the columns beyond P + 1 || [hi] factor P + 1 -> ...  Fork / join by events (capturable).  The
// stream and events are created once per device and live for the process; a mutex serialises the enqueue.
struct SolveSide {
  cudaStream_t hi = nullptr;
  cudaEvent_t ev_main = nullptr, ev_hi = nullptr;
  bool ready = false;
};
static std::mutex g_solve_mutex;
static SolveSide g_solve_side[64];

static int solve_side(SolveSide** out) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return QMLL_ERR_CUDA;
  SolveSide& s = g_solve_side[dev];
  if (!s.ready) {
    int lo = 0, hi = 0;
    if (cudaDeviceGetStreamPriorityRange(&lo, &hi) != cudaSuccess) return QMLL_ERR_CUDA;
    if (cudaStreamCreateWithPriority(&s.hi, cudaStreamNonBlocking, hi) != cudaSuccess) return QMLL_ERR_CUDA;
    if (cudaEventCreateWithFlags(&s.ev_main, cudaEventDisableTiming) != cudaSuccess) return QMLL_ERR_CUDA;
    if (cudaEventCreateWithFlags(&s.ev_hi, cudaEventDisableTiming) != cudaSuccess) return QMLL_ERR_CUDA;
    if (cudaFuncSetAttribute(syrk_update_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kUSmemBytes) != cudaSuccess)
      return QMLL_ERR_CUDA;
    if (cudaFuncSetAttribute(trsv_back_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kTrsvSmemBytes) != cudaSuccess)
      return QMLL_ERR_CUDA;
    s.ready = true;
  }
  *out = &s;
  return QMLL_OK;
}

#define QMLL_SOLVE_CUDA(call) do { if ((call) != cudaSuccess) return QMLL_ERR_CUDA; } while (0)

// 64-wide steps over the 256-wide panel at K0; their updates touch the panel's own columns only
static int solve_factor_panel(double* M, int D, int ld, int K0, int32_t* info, cudaStream_t st) {
  const int n_rows = D + 1;
  const int nb2 = D - K0 < kNB2 ? D - K0 : kNB2;
  for (int k0 = K0; k0 < K0 + nb2; k0 += kNB) {
    const int nb = K0 + nb2 - k0 < kNB ? K0 + nb2 - k0 : kNB;
    potrf_diag_kernel<<<1, 256, 0, st>>>(M, ld, k0, nb, info);
    QMLL_LAUNCH_CHECK("potrf_diag_kernel");
    const int rest = n_rows - k0 - nb;                    // >= 1: the right-hand side row
    trsm_panel_kernel<<<(rest + 127) / 128, 128, 0, st>>>(M, n_rows, ld, k0, nb);
    QMLL_LAUNCH_CHECK("trsm_panel_kernel");
    const int c0 = k0 + nb, c1 = K0 + nb2;               // the panel's remaining columns
    if (c1 > c0) {
      dim3 g((unsigned)((n_rows - c0 + kUM - 1) / kUM), (unsigned)((c1 - c0 + kUN - 1) / kUN));
      syrk_update_kernel<<<g, 128, kUSmemBytes, st>>>(M, n_rows, ld, c0, c0, c1, k0, nb);
      QMLL_LAUNCH_CHECK("syrk_update_kernel(panel)");
    }
  }
  return QMLL_OK;
}

int solve_normal_equations(const float* ZtZ, const float* Zty, int32_t D, double lambda, float* alpha, int32_t* info,
                           void* ws_ptr, size_t ws_bytes, cudaStream_t st) {
  if (D > 65534) return QMLL_ERR_UNSUPPORTED;             // grid.y of the prepare pass; 34 GB of FP64 beyond that
  const int ld = solve_ld(D), n_rows = D + 1;
  Carver ws(ws_ptr, ws_bytes);
  double* M = ws.take<double>((size_t)(D + 2) * ld);
  double* sol = ws.take<double>((size_t)D);
  const int n_blk = (D + kNB - 1) / kNB;
  int* flags = ws.take<int>((size_t)n_blk + 1);            // [n_blk] block-solved flags + the CTA ticket
  if (!ws_ptr || ((uintptr_t)ws_ptr & 255) != 0 || !ws.fits()) return QMLL_ERR_WORKSPACE;
  std::lock_guard<std::mutex> lock(g_solve_mutex);
  SolveSide* side = nullptr;
  if (int rc = solve_side(&side)) return rc;
  cudaStream_t hi = side->hi;
  double* y = M + (size_t)D * ld;                           // row D: b on entry, y = L^-1 b after the factorisation
  solve_prepare_kernel<<<dim3((unsigned)((D + 1023) / 1024), (unsigned)(D + 1)), 256, 0, st>>>(ZtZ, Zty, D, ld, lambda, M, y, info, flags, n_blk + 1);
  QMLL_LAUNCH_CHECK("solve_prepare_kernel");
  QMLL_SOLVE_CUDA(cudaEventRecord(side->ev_main, st));
  QMLL_SOLVE_CUDA(cudaStreamWaitEvent(hi, side->ev_main, 0));
  if (int rc = solve_factor_panel(M, D, ld, 0, info, hi)) return rc;
  for (int K0 = 0; K0 < D; K0 += kNB2) {
    const int nb2 = D - K0 < kNB2 ? D - K0 : kNB2;
    const int t0 = K0 + nb2;                                // trailing matrix starts here
    if (t0 >= D) break;
    const int t1 = D - t0 < kNB2 ? D : t0 + kNB2;           // end of the next panel's columns
    {                                                       // [hi] columns of the next panel only
      dim3 g((unsigned)((n_rows - t0 + kUM - 1) / kUM), (unsigned)((t1 - t0 + kUN - 1) / kUN));
      syrk_update_kernel<<<g, 128, kUSmemBytes, hi>>>(M, n_rows, ld, t0, t0, t1, K0, nb2);
      QMLL_LAUNCH_CHECK("syrk_update_kernel(look-ahead)");
    }
    QMLL_SOLVE_CUDA(cudaEventRecord(side->ev_hi, hi));
    QMLL_SOLVE_CUDA(cudaStreamWaitEvent(st, side->ev_hi, 0));
    if (t1 < D) {                                           // [caller] the rest of the trailing matrix
      dim3 g((unsigned)((n_rows - t1 + kUM - 1) / kUM), (unsigned)((D - t1 + kUN - 1) / kUN));
      syrk_update_kernel<<<g, 128, kUSmemBytes, st>>>(M, n_rows, ld, t1, t1, D, K0, nb2);
      QMLL_LAUNCH_CHECK("syrk_update_kernel(trailing)");
    }
    QMLL_SOLVE_CUDA(cudaEventRecord(side->ev_main, st));
    if (int rc = solve_factor_panel(M, D, ld, t0, info, hi)) return rc;   // [hi] overlaps the trailing update
    QMLL_SOLVE_CUDA(cudaStreamWaitEvent(hi, side->ev_main, 0));           // before hi touches columns >= t1
  }
  QMLL_SOLVE_CUDA(cudaEventRecord(side->ev_hi, hi));
  QMLL_SOLVE_CUDA(cudaStreamWaitEvent(st, side->ev_hi, 0));
  trsv_back_kernel<<<(D + 127) / 128, 128, kTrsvSmemBytes, st>>>(M, D, ld, y, sol, flags, flags + n_blk);   // L^T alpha = y
  QMLL_LAUNCH_CHECK("trsv_back_kernel");
  solve_finish_kernel<<<(D + 255) / 256, 256, 0, st>>>(sol, alpha, D);
  QMLL_LAUNCH_CHECK("solve_finish_kernel");
  return QMLL_OK;
}

}  // namespace qmll
