// solve_kernels.cu -- NEXT #1 of SURVEY.md section 8(f): alpha = (ZtZ + lambda I)^-1 Zty  (eq. 16-17;
// "solved by LU decomposition", L137 -- the matrix is symmetric positive definite, so Cholesky).  FP64 throughout: the
// Gram matrix of random features is ill-conditioned (the paper's FP32 round-off remark, L351), and the O(D^3/3) solve
// is small beside the O(rows D^2) accumulation.  Two-level blocked right-looking Cholesky:
//   potrf_diag_kernel (one CTA, 64 x 64 diagonal block in shared memory)  ->  trsm_panel_kernel (thread per row)
//   ->  syrk_update_kernel on the 256-wide panel's own columns; after the panel one rank-256 syrk_update_kernel of
//   the trailing matrix (128 x 128 tiles, 8 x 8 DFMA register tiles),
// then forward / backward substitution by blocks.  `info` (device int) follows LAPACK: 0 = success, k > 0 = the
// leading minor of order k is not positive definite (the factorisation then carries NaNs).
#include "qmll_common.cuh"

namespace qmll {

constexpr int kNB = 64;     // inner step: diagonal block factorised in shared memory
constexpr int kNB2 = 256;   // outer panel: one trailing update per 256 columns

__global__ void solve_prepare_kernel(const float* __restrict__ ZtZ, const float* __restrict__ Zty, int D, double lambda,
                                     double* __restrict__ M, double* __restrict__ rhs, int* __restrict__ info) {
  const long long n = (long long)D * D;
  for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < n;
       idx += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(idx / D), j = (int)(idx % D);
    M[idx] = (double)ZtZ[idx] + (i == j ? lambda : 0.0);
    if (j == 0) rhs[i] = (double)Zty[i];
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) *info = 0;
}

// Cholesky of the nb x nb diagonal block at (k0, k0): A = L L^T, L overwrites the lower triangle.
__global__ void __launch_bounds__(256) potrf_diag_kernel(double* __restrict__ M, int D, int k0, int nb, int* info) {
  __shared__ double a[kNB][kNB + 1];
  const int t = threadIdx.x;
  for (int idx = t; idx < nb * nb; idx += 256) a[idx / nb][idx % nb] = M[(size_t)(k0 + idx / nb) * D + k0 + idx % nb];
  __syncthreads();
  for (int j = 0; j < nb; ++j) {
    const double piv = a[j][j];
    __syncthreads();
    if (t == 0) {
      if (!(piv > 0.0) && *info == 0) *info = k0 + j + 1;
      a[j][j] = sqrt(piv);
    }
    __syncthreads();
    const double dinv = 1.0 / a[j][j];
    for (int i = j + 1 + t; i < nb; i += 256) a[i][j] *= dinv;
    __syncthreads();
    // trailing update of the lower triangle: a[i][c] -= a[i][j] * a[c][j],  j < c <= i < nb
    const int m = nb - j - 1;
    for (int idx = t; idx < m * m; idx += 256) {
      const int i = j + 1 + idx / m, c = j + 1 + idx % m;
      if (c <= i) a[i][c] -= a[i][j] * a[c][j];
    }
    __syncthreads();
  }
  for (int idx = t; idx < nb * nb; idx += 256) {
    const int i = idx / nb, c = idx % nb;
    if (c <= i) M[(size_t)(k0 + i) * D + k0 + c] = a[i][c];
  }
}

// Rows below the diagonal block: X = A21 L11^-T, one thread per row (forward substitution along the row).
__global__ void __launch_bounds__(128) trsm_panel_kernel(double* __restrict__ M, int D, int k0, int nb) {
  __shared__ double l[kNB][kNB + 1];
  for (int idx = threadIdx.x; idx < nb * nb; idx += 128) l[idx / nb][idx % nb] = M[(size_t)(k0 + idx / nb) * D + k0 + idx % nb];
  __syncthreads();
  const int i = k0 + nb + blockIdx.x * 128 + threadIdx.x;
  if (i >= D) return;
  double* row = M + (size_t)i * D + k0;
  double x[kNB];
#pragma unroll
  for (int c = 0; c < kNB; ++c) x[c] = c < nb ? row[c] : 0.0;
#pragma unroll
  for (int c = 0; c < kNB; ++c) {
    if (c < nb) {
      double s = x[c];
#pragma unroll
      for (int m = 0; m < c; ++m) s = fma(-x[m], l[c][m], s);
      x[c] = s / l[c][c];
    }
  }
#pragma unroll
  for (int c = 0; c < kNB; ++c)
    if (c < nb) row[c] = x[c];
}

// Symmetric rank-kn update on the lower triangle:  C[i][j] -= sum_{m < kn} M[i][k0 + m] * M[j][k0 + m]  for rows
// i >= r0, columns c0 <= j < c1, j <= i.  CTA = 128 x 128 tile (blockIdx.x: row tile from r0, blockIdx.y: column tile
// from c0), thread = 8 x 8 outputs (rows ty + 16 u, columns tx + 16 v: shared-memory reads are broadcasts or
// conflict-free, the write-back is coalesced), k in chunks of 16 through shared memory.  64 DFMA per 16 LDS.64: the
// FP64 pipe, not shared memory, bounds it.
constexpr int kUT = 128;   // tile
constexpr int kUK = 16;    // k chunk
__global__ void __launch_bounds__(256) syrk_update_kernel(double* __restrict__ M, int D, int r0, int c0, int c1, int k0,
                                                          int kn) {
  const int i0 = r0 + blockIdx.x * kUT, j0 = c0 + blockIdx.y * kUT;
  if (j0 >= c1 || j0 > i0 + kUT - 1) return;          // tile entirely above the diagonal or outside the column range
  __shared__ double li[kUK][kUT + 2], lj[kUK][kUT + 2];
  const int t = threadIdx.x, tx = t & 15, ty = t >> 4;
  double acc[8][8];
#pragma unroll
  for (int u = 0; u < 8; ++u)
#pragma unroll
    for (int v = 0; v < 8; ++v) acc[u][v] = 0.0;
  // 128 rows x 16 k doubles per operand and chunk: thread t owns row t / 2, k half t % 2 (8 doubles = 64 contiguous
  // bytes).  The next chunk is fetched into registers while the current one is multiplied (software pipeline).
  const int lr = t >> 1, lkh = (t & 1) * 8;
  const bool oki = i0 + lr < D, okj = j0 + lr < D;
  const double* pi = M + (size_t)(oki ? i0 + lr : 0) * D + k0 + lkh;
  const double* pj = M + (size_t)(okj ? j0 + lr : 0) * D + k0 + lkh;
  double ni[8], nj[8];
  auto fetch = [&](int m0) {
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      const bool okm = m0 + lkh + q < kn;
      ni[q] = (oki && okm) ? pi[m0 + q] : 0.0;
      nj[q] = (okj && okm) ? pj[m0 + q] : 0.0;
    }
  };
  fetch(0);
  for (int m0 = 0; m0 < kn; m0 += kUK) {
    __syncthreads();
#pragma unroll
    for (int q = 0; q < 8; ++q) { li[lkh + q][lr] = ni[q]; lj[lkh + q][lr] = nj[q]; }
    __syncthreads();
    if (m0 + kUK < kn) fetch(m0 + kUK);
#pragma unroll
    for (int m = 0; m < kUK; ++m) {
      double a[8], b[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) { a[u] = li[m][ty + 16 * u]; b[u] = lj[m][tx + 16 * u]; }
#pragma unroll
      for (int u = 0; u < 8; ++u)
#pragma unroll
        for (int v = 0; v < 8; ++v) acc[u][v] = fma(a[u], b[v], acc[u][v]);
    }
  }
#pragma unroll
  for (int u = 0; u < 8; ++u)
#pragma unroll
    for (int v = 0; v < 8; ++v) {
      const int i = i0 + ty + 16 * u, j = j0 + tx + 16 * v;
      if (i < D && j < c1 && j <= i) M[(size_t)i * D + j] -= acc[u][v];
    }
}

// Substitution, diagonal block: transposed = 0 solves L11 y = b (forward), 1 solves L11^T a = y (backward).
__global__ void __launch_bounds__(64) trsv_diag_kernel(const double* __restrict__ M, int D, int k0, int nb, int transposed,
                                                       double* __restrict__ rhs) {
  __shared__ double l[kNB][kNB + 1];
  __shared__ double b[kNB];
  const int t = threadIdx.x;
  for (int idx = t; idx < nb * nb; idx += 64) l[idx / nb][idx % nb] = M[(size_t)(k0 + idx / nb) * D + k0 + idx % nb];
  if (t < nb) b[t] = rhs[k0 + t];
  __syncthreads();
  if (!transposed) {
    for (int c = 0; c < nb; ++c) {
      if (t == c) b[c] /= l[c][c];
      __syncthreads();
      if (t > c && t < nb) b[t] -= l[t][c] * b[c];
      __syncthreads();
    }
  } else {
    for (int c = nb - 1; c >= 0; --c) {
      if (t == c) b[c] /= l[c][c];
      __syncthreads();
      if (t < c) b[t] -= l[c][t] * b[c];
      __syncthreads();
    }
  }
  if (t < nb) rhs[k0 + t] = b[t];
}

// Forward: rhs[i] -= sum_m L[i][k0+m] y[k0+m] for i >= k0+nb.  Backward: rhs[j] -= sum_m L[k0+m][j] a[k0+m] for j < k0.
__global__ void __launch_bounds__(128) trsv_update_kernel(const double* __restrict__ M, int D, int k0, int nb,
                                                          int transposed, double* __restrict__ rhs) {
  __shared__ double y[kNB];
  if (threadIdx.x < nb) y[threadIdx.x] = rhs[k0 + threadIdx.x];
  __syncthreads();
  const int idx = blockIdx.x * 128 + threadIdx.x;
  if (!transposed) {
    const int i = k0 + nb + idx;
    if (i >= D) return;
    const double* row = M + (size_t)i * D + k0;
    double s = 0.0;
    for (int m = 0; m < nb; ++m) s = fma(row[m], y[m], s);
    rhs[i] -= s;
  } else {
    const int j = idx;
    if (j >= k0) return;
    double s = 0.0;
    for (int m = 0; m < nb; ++m) s = fma(M[(size_t)(k0 + m) * D + j], y[m], s);
    rhs[j] -= s;
  }
}

__global__ void solve_finish_kernel(const double* __restrict__ rhs, float* __restrict__ alpha, int D) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < D) alpha[i] = (float)rhs[i];
}

size_t solve_workspace_bytes(int32_t D) { return align_up((size_t)D * D * 8, 256) + align_up((size_t)D * 8, 256) + 512; }

int solve_normal_equations(const float* ZtZ, const float* Zty, int32_t D, double lambda, float* alpha, int32_t* info,
                           void* ws_ptr, size_t ws_bytes, cudaStream_t st) {
  Carver ws(ws_ptr, ws_bytes);
  double* M = ws.take<double>((size_t)D * D);
  double* rhs = ws.take<double>((size_t)D);
  if (!ws_ptr || ((uintptr_t)ws_ptr & 255) != 0 || !ws.fits()) return QMLL_ERR_WORKSPACE;
  solve_prepare_kernel<<<1184, 256, 0, st>>>(ZtZ, Zty, D, lambda, M, rhs, info);
  QMLL_LAUNCH_CHECK("solve_prepare_kernel");
  // Two levels: 64-wide steps factor a 256-wide panel (their updates touch the panel's own columns only), then ONE
  // rank-256 update of the trailing matrix: the trailing matrix is read and written D / 256 times instead of D / 64.
  for (int K0 = 0; K0 < D; K0 += kNB2) {
    const int nb2 = D - K0 < kNB2 ? D - K0 : kNB2;
    for (int k0 = K0; k0 < K0 + nb2; k0 += kNB) {
      const int nb = K0 + nb2 - k0 < kNB ? K0 + nb2 - k0 : kNB;
      potrf_diag_kernel<<<1, 256, 0, st>>>(M, D, k0, nb, info);
      QMLL_LAUNCH_CHECK("potrf_diag_kernel");
      const int rest = D - k0 - nb;
      if (rest > 0) {
        trsm_panel_kernel<<<(rest + 127) / 128, 128, 0, st>>>(M, D, k0, nb);
        QMLL_LAUNCH_CHECK("trsm_panel_kernel");
        const int c0 = k0 + nb, c1 = K0 + nb2;             // the panel's remaining columns
        if (c1 > c0) {
          dim3 g((unsigned)((D - c0 + kUT - 1) / kUT), (unsigned)((c1 - c0 + kUT - 1) / kUT));
          syrk_update_kernel<<<g, 256, 0, st>>>(M, D, c0, c0, c1, k0, nb);
          QMLL_LAUNCH_CHECK("syrk_update_kernel(panel)");
        }
      }
    }
    const int t0 = K0 + nb2;                                // trailing matrix
    if (t0 < D) {
      const unsigned nt = (unsigned)((D - t0 + kUT - 1) / kUT);
      syrk_update_kernel<<<dim3(nt, nt), 256, 0, st>>>(M, D, t0, t0, D, K0, nb2);
      QMLL_LAUNCH_CHECK("syrk_update_kernel(trailing)");
    }
  }
  for (int k0 = 0; k0 < D; k0 += kNB) {  // L y = b
    const int nb = D - k0 < kNB ? D - k0 : kNB;
    trsv_diag_kernel<<<1, 64, 0, st>>>(M, D, k0, nb, 0, rhs);
    QMLL_LAUNCH_CHECK("trsv_diag_kernel");
    const int rest = D - k0 - nb;
    if (rest > 0) {
      trsv_update_kernel<<<(rest + 127) / 128, 128, 0, st>>>(M, D, k0, nb, 0, rhs);
      QMLL_LAUNCH_CHECK("trsv_update_kernel");
    }
  }
  for (int k0 = (D - 1) / kNB * kNB; k0 >= 0; k0 -= kNB) {  // L^T alpha = y
    const int nb = D - k0 < kNB ? D - k0 : kNB;
    trsv_diag_kernel<<<1, 64, 0, st>>>(M, D, k0, nb, 1, rhs);
    QMLL_LAUNCH_CHECK("trsv_diag_kernel");
    if (k0 > 0) {
      trsv_update_kernel<<<(k0 + 127) / 128, 128, 0, st>>>(M, D, k0, nb, 1, rhs);
      QMLL_LAUNCH_CHECK("trsv_update_kernel");
    }
  }
  solve_finish_kernel<<<(D + 255) / 256, 256, 0, st>>>(rhs, alpha, D);
  QMLL_LAUNCH_CHECK("solve_finish_kernel");
  return QMLL_OK;
}

}  // namespace qmll
