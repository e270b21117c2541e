// solve_kernels.cu -- NEXT #1 of SURVEY.md section 8(f): alpha = (ZtZ + lambda I)^-1 Zty  (eq. 16-17;
// "solved by LU decomposition", L137 -- the matrix is symmetric positive definite, so Cholesky).  FP64 throughout: the
// Gram matrix of random features is ill-conditioned (the paper's FP32 round-off remark, L351), and the O(D^3/3) solve
// is small beside the O(rows D^2) accumulation.  Blocked right-looking Cholesky (64-wide panels):
//   potrf_diag_kernel (one CTA, diagonal block in shared memory)  ->  trsm_panel_kernel (thread per row)
//   ->  syrk_update_kernel (64 x 64 x 64 DFMA tiles over the lower triangle of the trailing matrix),
// then forward / backward substitution by blocks.  `info` (device int) follows LAPACK: 0 = success, k > 0 = the
// leading minor of order k is not positive definite (the factorisation then carries NaNs).
#include "qmll_common.cuh"

namespace qmll {

constexpr int kNB = 64;

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

// Trailing update A22 -= L21 L21^T on the lower triangle: CTA (ti, tj), tj <= ti, computes a 64 x 64 tile.
__global__ void __launch_bounds__(256) syrk_update_kernel(double* __restrict__ M, int D, int k0, int nb) {
  if (blockIdx.y > blockIdx.x) return;
  __shared__ double li[64][33], lj[64][33];  // one half of the 64-wide panel at a time (static smem <= 48 KB)
  const int base = k0 + nb;
  const int i0 = base + blockIdx.x * 64, j0 = base + blockIdx.y * 64;
  const int t = threadIdx.x;
  const int tr = (t / 16) * 4, tc = (t % 16) * 4;  // 4 x 4 outputs per thread
  double acc[4][4] = {};
  for (int mh = 0; mh < kNB; mh += 32) {
    __syncthreads();
    for (int idx = t; idx < 64 * 32; idx += 256) {
      const int r = idx / 32, m = mh + idx % 32;
      li[r][idx % 32] = (i0 + r < D && m < nb) ? M[(size_t)(i0 + r) * D + k0 + m] : 0.0;
      lj[r][idx % 32] = (j0 + r < D && m < nb) ? M[(size_t)(j0 + r) * D + k0 + m] : 0.0;
    }
    __syncthreads();
#pragma unroll 8
    for (int m = 0; m < 32; ++m) {
      double a[4], b[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) { a[u] = li[tr + u][m]; b[u] = lj[tc + u][m]; }
#pragma unroll
      for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int v = 0; v < 4; ++v) acc[u][v] = fma(a[u], b[v], acc[u][v]);
    }
  }
#pragma unroll
  for (int u = 0; u < 4; ++u)
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      const int i = i0 + tr + u, j = j0 + tc + v;
      if (i < D && j <= i) M[(size_t)i * D + j] -= acc[u][v];
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
  for (int k0 = 0; k0 < D; k0 += kNB) {
    const int nb = D - k0 < kNB ? D - k0 : kNB;
    potrf_diag_kernel<<<1, 256, 0, st>>>(M, D, k0, nb, info);
    QMLL_LAUNCH_CHECK("potrf_diag_kernel");
    const int rest = D - k0 - nb;
    if (rest > 0) {
      trsm_panel_kernel<<<(rest + 127) / 128, 128, 0, st>>>(M, D, k0, nb);
      QMLL_LAUNCH_CHECK("trsm_panel_kernel");
      const unsigned nt = (unsigned)((rest + 63) / 64);
      syrk_update_kernel<<<dim3(nt, nt), 256, 0, st>>>(M, D, k0, nb);
      QMLL_LAUNCH_CHECK("syrk_update_kernel");
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
