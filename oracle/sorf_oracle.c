/* oracle/sorf_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, FP64 CPU statement of what the SORF hot path of QML-Lightning computes
 * (arXiv 2206.01580; citations are PAPER.md line numbers + equation).  It follows the
 * paper's algorithm step by step, in the paper's order: no blocking, no fusion, no
 * reordering.  It shares no code, header, table or helper with the CUDA path under
 * paper_2206_01580_b200/ and neither side includes the other.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Inputs are the same fp32 / int8 / int32 arrays the GPU library receives, widened to
 * double on read.  All outputs are double.
 *
 * Readings of the paper where it is silent or garbled (SURVEY.md
 * section 8(c) A1-A16):
 *   A2  each H in eq. 20 is implicitly orthonormal: with the unnormalised Sylvester matrix
 *       used here the constant is  c = (sqrt(d)/sigma) * d^(-T/2).
 *   A3  H in natural (Hadamard) order, H[i][j] = (-1)^popcount(i & j)  (recursion L163-165).
 *   A4  sign flip first, then H; signs[., ., t=0, .] is D_1 and multiplies x (L268).
 *   A5  feature index l = s*d + m (stack-major concatenation, L167).
 *   A6  sign diagonals AND b are per element (BASELINE.json).
 *   A8  force rows are G = -dZ/dr so that [Z; G] alpha = [E; F]  (F = -dE/dr, eq. 5/10 L63, L90).
 *   A12 dense gradient of molecule M with n atoms: [n, d, n, 3] = (I, m, j, k) = dx_I[m]/dr_{j,k}.
 *   A13 neighbour gradient: entry (I, q) is dx_I/dr_j with j = nbr_idx[I, q]; duplicates and
 *       self indices accumulate; -1 is padding.
 *
 * Pins (tests/test_oracle_pins.py): explicit dense H from the recursion, H*H = d*I, the
 * all-plus-signs closed form, the per-stack norm invariant, Monte-Carlo convergence to the
 * Gaussian kernel, a dense-W brute force of eq. 14/15, finite-difference forces, G*alpha = F,
 * finite differences of Z against G, Gram-matrix identities and a BLAS cross-check, and
 * sparse == scattered-dense gradients; qo_project: numpy matmul, the identity U^T U = I (columns of U_e project
 * onto unit vectors), the norm inequality |x| <= |rho| with equality on the span, and finite differences of a
 * smooth rho(r) for the projected gradient.  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int qo_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* In-place unnormalised Walsh-Hadamard transform, natural order: v <- H_d v with
 * H_{2^n} = [[H, H], [H, -H]], H_1 = 1.  Textbook iterative butterfly
 * ("fast Hadamard transform using in-place operations in O(d log d)", L167). */
void qo_fwht(double* v, int d) {
  for (int h = 1; h < d; h <<= 1)
    for (int i = 0; i < d; i += 2 * h)
      for (int j = i; j < i + h; ++j) {
        double a = v[j], b = v[j + h];
        v[j] = a + b;
        v[j + h] = a - b;
      }
}

/* c = sqrt(d)/sigma * d^(-T/2): eq. 20 (L158) with each H orthonormal (reading A2). */
double qo_scale(int d, int T, double sigma) {
  return sqrt((double)d) / sigma * pow((double)d, -0.5 * (double)T);
}

/* One stack of the SORF linear map applied to an arbitrary column `col` (length d):
 *   v <- col;  for t = 0..T-1:  v <- H (S[e,s,t,:] .* v);   out <- c * v
 * eq. 20 L158-161 and L268 ("after multiplication with the diagonal sign flipping matrix"). */
static void chain_forward(const double* col, const int8_t* S_es /* [T, d] */, int d, int T, double c,
                          double* out) {
  for (int m = 0; m < d; ++m) out[m] = col[m];
  for (int t = 0; t < T; ++t) {
    const int8_t* S = S_es + (size_t)t * d;
    for (int m = 0; m < d; ++m) out[m] *= (double)S[m];
    qo_fwht(out, d);
  }
  for (int m = 0; m < d; ++m) out[m] *= c;
}

/* Transposed map of one stack: (c H D_T ... H D_1)^T q = c D_1 H ... D_T H q  (H symmetric):
 *   v <- q;  for t = T-1..0:  v <- S[e,s,t,:] .* (H v);   out <- c * v */
static void chain_transposed(const double* q, const int8_t* S_es, int d, int T, double c, double* out) {
  for (int m = 0; m < d; ++m) out[m] = q[m];
  for (int t = T - 1; t >= 0; --t) {
    const int8_t* S = S_es + (size_t)t * d;
    qo_fwht(out, d);
    for (int m = 0; m < d; ++m) out[m] *= (double)S[m];
  }
  for (int m = 0; m < d; ++m) out[m] *= c;
}

/* u[l] = (W_e x)[l],  l = s*d + m, for one atom (eq. 20; concatenation of D/d stacks, L167). */
void qo_sorf_u(const float* x_I, int e, int d, int D, int T, double sigma, const int8_t* signs,
               double* u /* [D] */) {
  const int n_s = D / d;
  const double c = qo_scale(d, T, sigma);
  double* col = (double*)malloc(sizeof(double) * d);
  for (int m = 0; m < d; ++m) col[m] = (double)x_I[m];
  for (int s = 0; s < n_s; ++s)
    chain_forward(col, signs + ((size_t)e * n_s + s) * T * d, d, T, c, u + (size_t)s * d);
  free(col);
}

/* Z[M, l] = sum_{I in M} sqrt(2/D) cos(u_I[l] + b[e_I, l])   (eq. 14, eq. 15). */
void qo_forward(const float* x, const int32_t* elem, const int32_t* mol_off, int64_t n_atoms, int n_mol,
                int d, int D, int T, double sigma, const int8_t* signs, const float* bias,
                double* Z /* [n_mol, D] */) {
  (void)n_atoms;
  const double nrm = sqrt(2.0 / (double)D);
#pragma omp parallel for schedule(dynamic, 1)
  for (int M = 0; M < n_mol; ++M) {
    double* u = (double*)malloc(sizeof(double) * D);
    double* zrow = Z + (size_t)M * D;
    for (int l = 0; l < D; ++l) zrow[l] = 0.0;
    for (int64_t I = mol_off[M]; I < mol_off[M + 1]; ++I) {
      const int e = elem[I];
      qo_sorf_u(x + (size_t)I * d, e, d, D, T, sigma, signs, u);
      for (int l = 0; l < D; ++l) zrow[l] += nrm * cos(u[l] + (double)bias[(size_t)e * D + l]);
    }
    free(u);
  }
}

/* E_M = sum_l Z[M, l] alpha[l]   (eq. 15). */
void qo_energy(const double* Z, const float* alpha, int n_mol, int D, double* energy) {
  for (int M = 0; M < n_mol; ++M) {
    double acc = 0.0;
    for (int l = 0; l < D; ++l) acc += Z[(size_t)M * D + l] * (double)alpha[l];
    energy[M] = acc;
  }
}

/* g_I = dE/dx_I: chain rule through eq. 14 and eq. 20.
 *   q[l] = -sqrt(2/D) alpha[l] sin(u[l] + b[e,l]);  g_I = sum_s W_{e,s}^T q_s. */
void qo_backward_g(const float* x, const int32_t* elem, int64_t n_atoms, int d, int D, int T, double sigma,
                   const int8_t* signs, const float* bias, const float* alpha, double* g /* [n_atoms, d] */) {
  const int n_s = D / d;
  const double nrm = sqrt(2.0 / (double)D);
  const double c = qo_scale(d, T, sigma);
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t I = 0; I < n_atoms; ++I) {
    double* u = (double*)malloc(sizeof(double) * D);
    double* q = (double*)malloc(sizeof(double) * d);
    double* v = (double*)malloc(sizeof(double) * d);
    const int e = elem[I];
    qo_sorf_u(x + (size_t)I * d, e, d, D, T, sigma, signs, u);
    double* gI = g + (size_t)I * d;
    for (int m = 0; m < d; ++m) gI[m] = 0.0;
    for (int s = 0; s < n_s; ++s) {
      for (int m = 0; m < d; ++m) {
        const int l = s * d + m;
        q[m] = -nrm * (double)alpha[l] * sin(u[l] + (double)bias[(size_t)e * D + l]);
      }
      chain_transposed(q, signs + ((size_t)e * n_s + s) * T * d, d, T, c, v);
      for (int m = 0; m < d; ++m) gI[m] += v[m];
    }
    free(u); free(q); free(v);
  }
}

/* F[j,k] = - sum_I sum_m g_I[m] dx_I[m]/dr_{j,k}   (F = -dE/dr, eq. 5/10 L63, L90), dense layout A12:
 * molecule M with n atoms owns the block [n, d, n, 3] at dense + dense_off[M]. */
void qo_forces_dense(const double* g, const int32_t* mol_off, int n_mol, int d, const float* dense,
                     const int64_t* dense_off, double* F /* [n_atoms, 3] */) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int M = 0; M < n_mol; ++M) {
    const int64_t a0 = mol_off[M];
    const int n = mol_off[M + 1] - mol_off[M];
    const float* dx = dense + dense_off[M];
    for (int j = 0; j < n; ++j)
      for (int k = 0; k < 3; ++k) {
        double acc = 0.0;
        for (int I = 0; I < n; ++I)
          for (int m = 0; m < d; ++m)
            acc += g[(size_t)(a0 + I) * d + m] * (double)dx[(((size_t)I * d + m) * n + j) * 3 + k];
        F[(size_t)(a0 + j) * 3 + k] = -acc;
      }
  }
}

/* Same contraction, neighbour-sparse layout A13 (serial: duplicates accumulate in index order). */
void qo_forces_neighbor(const double* g, int64_t n_atoms, int d, int K, const int32_t* nbr_idx,
                        const float* nbr_val, double* F /* [n_atoms, 3] */) {
  for (int64_t i = 0; i < n_atoms * 3; ++i) F[i] = 0.0;
  for (int64_t I = 0; I < n_atoms; ++I)
    for (int q = 0; q < K; ++q) {
      const int32_t j = nbr_idx[(size_t)I * K + q];
      if (j < 0) continue;
      const float* val = nbr_val + ((size_t)I * K + q) * d * 3;
      for (int k = 0; k < 3; ++k) {
        double acc = 0.0;
        for (int m = 0; m < d; ++m) acc += g[(size_t)I * d + m] * (double)val[(size_t)m * 3 + k];
        F[(size_t)j * 3 + k] -= acc;
      }
    }
}

/* Force rows (derivative features, L137; sign reading A8):
 *   G[(j,k), l] = - dZ[M,l]/dr_{j,k} = + sum_{I in M} sqrt(2/D) sin(u_I[l] + b[e_I,l]) (W_{e_I} dx_I[:,j,k])[l]
 * rows ordered (M, atom j, k) = 3*(global atom index j) + k.  Dense layout. */
void qo_force_rows_dense(const float* x, const int32_t* elem, const int32_t* mol_off, int n_mol, int d, int D,
                         int T, double sigma, const int8_t* signs, const float* bias, const float* dense,
                         const int64_t* dense_off, double* G /* [3 n_atoms, D] */) {
  const int n_s = D / d;
  const double nrm = sqrt(2.0 / (double)D);
  const double c = qo_scale(d, T, sigma);
#pragma omp parallel for schedule(dynamic, 1)
  for (int M = 0; M < n_mol; ++M) {
    const int64_t a0 = mol_off[M];
    const int n = mol_off[M + 1] - mol_off[M];
    const float* dx = dense + dense_off[M];
    double* u = (double*)malloc(sizeof(double) * D);
    double* zs = (double*)malloc(sizeof(double) * D);
    double* col = (double*)malloc(sizeof(double) * d);
    double* w = (double*)malloc(sizeof(double) * d);
    for (int64_t r = 3 * a0; r < 3 * (a0 + n); ++r)
      for (int l = 0; l < D; ++l) G[(size_t)r * D + l] = 0.0;
    for (int I = 0; I < n; ++I) {
      const int e = elem[a0 + I];
      qo_sorf_u(x + (size_t)(a0 + I) * d, e, d, D, T, sigma, signs, u);
      for (int l = 0; l < D; ++l) zs[l] = nrm * sin(u[l] + (double)bias[(size_t)e * D + l]);
      for (int j = 0; j < n; ++j)
        for (int k = 0; k < 3; ++k) {
          for (int m = 0; m < d; ++m) col[m] = (double)dx[(((size_t)I * d + m) * n + j) * 3 + k];
          double* Grow = G + ((size_t)(a0 + j) * 3 + k) * D;
          for (int s = 0; s < n_s; ++s) {
            chain_forward(col, signs + ((size_t)e * n_s + s) * T * d, d, T, c, w);
            for (int m = 0; m < d; ++m) Grow[s * d + m] += zs[s * d + m] * w[m];
          }
        }
    }
    free(u); free(zs); free(col); free(w);
  }
}

/* Force rows, neighbour layout (serial over atoms: rows of different atoms collide). */
void qo_force_rows_neighbor(const float* x, const int32_t* elem, int64_t n_atoms, int d, int D, int T,
                            double sigma, const int8_t* signs, const float* bias, int K,
                            const int32_t* nbr_idx, const float* nbr_val, double* G /* [3 n_atoms, D] */) {
  const int n_s = D / d;
  const double nrm = sqrt(2.0 / (double)D);
  const double c = qo_scale(d, T, sigma);
  double* u = (double*)malloc(sizeof(double) * D);
  double* zs = (double*)malloc(sizeof(double) * D);
  double* col = (double*)malloc(sizeof(double) * d);
  double* w = (double*)malloc(sizeof(double) * d);
  for (size_t i = 0; i < (size_t)n_atoms * 3 * D; ++i) G[i] = 0.0;
  for (int64_t I = 0; I < n_atoms; ++I) {
    const int e = elem[I];
    qo_sorf_u(x + (size_t)I * d, e, d, D, T, sigma, signs, u);
    for (int l = 0; l < D; ++l) zs[l] = nrm * sin(u[l] + (double)bias[(size_t)e * D + l]);
    for (int q = 0; q < K; ++q) {
      const int32_t j = nbr_idx[(size_t)I * K + q];
      if (j < 0) continue;
      const float* val = nbr_val + ((size_t)I * K + q) * d * 3;
      for (int k = 0; k < 3; ++k) {
        for (int m = 0; m < d; ++m) col[m] = (double)val[(size_t)m * 3 + k];
        double* Grow = G + ((size_t)j * 3 + k) * D;
        for (int s = 0; s < n_s; ++s) {
          chain_forward(col, signs + ((size_t)e * n_s + s) * T * d, d, T, c, w);
          for (int m = 0; m < d; ++m) Grow[s * d + m] += zs[s * d + m] * w[m];
        }
      }
    }
  }
  free(u); free(zs); free(col); free(w);
}

/* Normal equations (eq. 16, eq. 17): ZtZ = A^T A, Zty = A^T y, the definition written out.
 * A is fp32 [rows, D] (what the GPU library is given), widened to double.  Every entry is the plain sum over
 * r = 0 .. rows-1 in that order; the row loop is the outer one only so that A is read along its rows (a thread
 * owns a block of rows i of ZtZ and visits A once). */
void qo_normal_equations(const float* A, const float* y, int64_t rows, int D, double* ZtZ /* [D, D] */,
                         double* Zty /* [D] */) {
#pragma omp parallel
  {
    int nt = 1, tid = 0;
#ifdef _OPENMP
    nt = omp_get_num_threads(); tid = omp_get_thread_num();
#endif
    const int i0 = (int)((int64_t)D * tid / nt), i1 = (int)((int64_t)D * (tid + 1) / nt);
    for (int i = i0; i < i1; ++i) {
      for (int j = 0; j < D; ++j) ZtZ[(size_t)i * D + j] = 0.0;
      Zty[i] = 0.0;
    }
    for (int64_t r = 0; r < rows; ++r) {
      const float* Ar = A + (size_t)r * D;
      for (int i = i0; i < i1; ++i) {
        const double a = (double)Ar[i];
        double* row = ZtZ + (size_t)i * D;
        for (int j = 0; j < D; ++j) row[j] += a * (double)Ar[j];
        Zty[i] += a * (double)y[r];
      }
    }
  }
}

/* Selected entries (i_k, j_k) of A^T A: the same definition, for sampled parity at full size. */
void qo_gram_entries(const float* A, int64_t rows, int D, const int32_t* ii, const int32_t* jj, int64_t n,
                     double* out) {
#pragma omp parallel
  {
    int nt = 1, tid = 0;
#ifdef _OPENMP
    nt = omp_get_num_threads(); tid = omp_get_thread_num();
#endif
    const int64_t k0 = n * tid / nt, k1 = n * (tid + 1) / nt;
    for (int64_t k = k0; k < k1; ++k) out[k] = 0.0;
    for (int64_t r = 0; r < rows; ++r) {
      const float* Ar = A + (size_t)r * D;
      for (int64_t k = k0; k < k1; ++k) out[k] += (double)Ar[ii[k]] * (double)Ar[jj[k]];
    }
  }
}

/* Selected full rows i_k of A^T A (out[k, :]), plus A^T y if y != NULL (out_y[k]). */
void qo_gram_rows(const float* A, const float* y, int64_t rows, int D, const int32_t* ii, int n,
                  double* out /* [n, D] */, double* out_y /* [n] or NULL */) {
#pragma omp parallel
  {
    int nt = 1, tid = 0;
#ifdef _OPENMP
    nt = omp_get_num_threads(); tid = omp_get_thread_num();
#endif
    const int j0 = (int)((int64_t)D * tid / nt), j1 = (int)((int64_t)D * (tid + 1) / nt);
    for (int k = 0; k < n; ++k)
      for (int j = j0; j < j1; ++j) out[(size_t)k * D + j] = 0.0;
    for (int64_t r = 0; r < rows; ++r) {
      const float* Ar = A + (size_t)r * D;
      for (int k = 0; k < n; ++k) {
        const double a = (double)Ar[ii[k]];
        double* row = out + (size_t)k * D;
        for (int j = j0; j < j1; ++j) row[j] += a * (double)Ar[j];
      }
    }
  }
  if (y && out_y) {
    for (int k = 0; k < n; ++k) {
      double acc = 0.0;
      for (int64_t r = 0; r < rows; ++r) acc += (double)A[(size_t)r * D + ii[k]] * (double)y[r];
      out_y[k] = acc;
    }
  }
}

/* Regularised normal equations (eq. 16-17): alpha = (ZtZ + lambda I)^-1 Zty.  The paper solves by LU (L137);
 * the matrix is symmetric positive definite, so this is the textbook (unblocked, row-by-row) Cholesky A = L L^T in
 * FP64 followed by the two triangular solves.  Returns 0, or k > 0 if the leading minor of order k is not positive
 * definite (LAPACK convention).  Pins: numpy.linalg.solve, residual, diagonal closed form, non-PD detection. */
int qo_solve(const float* ZtZ, const float* Zty, int D, double lambda, double* alpha /* [D] */) {
  double* L = (double*)malloc(sizeof(double) * (size_t)D * D);
  int info = 0;
  for (int i = 0; i < D && !info; ++i) {
    for (int j = 0; j <= i; ++j) {
      double s = (double)ZtZ[(size_t)i * D + j] + (i == j ? lambda : 0.0);
      for (int m = 0; m < j; ++m) s -= L[(size_t)i * D + m] * L[(size_t)j * D + m];
      if (i == j) {
        if (!(s > 0.0)) { info = i + 1; break; }
        L[(size_t)i * D + i] = sqrt(s);
      } else {
        L[(size_t)i * D + j] = s / L[(size_t)j * D + j];
      }
    }
  }
  if (!info) {
    for (int i = 0; i < D; ++i) {          /* L y = b */
      double s = (double)Zty[i];
      for (int m = 0; m < i; ++m) s -= L[(size_t)i * D + m] * alpha[m];
      alpha[i] = s / L[(size_t)i * D + i];
    }
    for (int i = D - 1; i >= 0; --i) {     /* L^T alpha = y */
      double s = alpha[i];
      for (int m = i + 1; m < D; ++m) s -= L[(size_t)m * D + i] * alpha[m];
      alpha[i] = s / L[(size_t)i * D + i];
    }
  }
  free(L);
  return info;
}

/* Per-element PCA projection (eq. 22): rho_I^proj = rho_I^T U_e^{N_PCA}, U_e^{N_PCA} = the first
 * N_PCA = d columns of the left singular vectors of eq. 21 for the element of atom I ("each element has its own
 * projection matrix").  U is [n_elem, rep, d] (the d kept columns), rho is [n_atoms, rep]:
 *   x[I, m] = sum_k rho[I, k] * U[e_I, k, m]. */
void qo_project(const float* rho, const int32_t* elem, int64_t n_atoms, int rep, int d, const float* U,
                double* x /* [n_atoms, d] */) {
#pragma omp parallel for schedule(static)
  for (int64_t I = 0; I < n_atoms; ++I) {
    const float* Ue = U + (size_t)elem[I] * rep * d;
    for (int m = 0; m < d; ++m) {
      double acc = 0.0;
      for (int k = 0; k < rep; ++k) acc += (double)rho[(size_t)I * rep + k] * (double)Ue[(size_t)k * d + m];
      x[(size_t)I * d + m] = acc;
    }
  }
}

/* The same projection applied to a dense descriptor gradient (U is constant, so d x_I / d r = (d rho_I / d r)^T U_e):
 * molecule M with n atoms holds [n, rep, n, 3] = (I, k, j, c) on input and [n, d, n, 3] = (I, m, j, c) on output
 * (layout A12 with rep resp. d as the descriptor length); in_off / out_off are the per-molecule float offsets. */
void qo_project_gradient(const float* gin, const int64_t* in_off, const int32_t* elem, const int32_t* mol_off,
                         int n_mol, int rep, int d, const float* U, const int64_t* out_off, double* gout) {
  for (int M = 0; M < n_mol; ++M) {
    const int a0 = mol_off[M], n = mol_off[M + 1] - a0, ncol = 3 * n;
    for (int I = 0; I < n; ++I) {
      const float* Ue = U + (size_t)elem[a0 + I] * rep * d;
      const float* src = gin + in_off[M] + (size_t)I * rep * ncol;
      double* dst = gout + out_off[M] + (size_t)I * d * ncol;
      for (int m = 0; m < d; ++m)
        for (int c = 0; c < ncol; ++c) {
          double acc = 0.0;
          for (int k = 0; k < rep; ++k) acc += (double)src[(size_t)k * ncol + c] * (double)Ue[(size_t)k * d + m];
          dst[(size_t)m * ncol + c] = acc;
        }
    }
  }
}

/* Random Fourier features with a DENSE matrix (eq. 12-14, eq. 18; the RFF arm of Fig. 1
 * L274-278), summed over the atoms of a molecule (eq. 15):
 *   Z[M, l] = sum_{I in M} sqrt(2/D) cos( sum_k W[e_I, l, k] x_I[k] + b[e_I, l] )
 * W [n_elem, D, d]: row l is w_l with the 1/sigma of eq. 18 already applied; per-element W and b as for SORF (A6).
 * Pins: the SORF oracle when W is the explicit dense SORF matrix (two code paths), numpy brute force, Monte-Carlo
 * convergence of z(x).z(y) to exp(-|x-y|^2 / 2 sigma^2) for Gaussian W (eq. 12-13). */
void qo_rff_forward(const float* W, const float* bias, int d, int D, const float* x, const int32_t* elem,
                    const int32_t* mol_off, int n_mol, double* Z /* [n_mol, D] */) {
  const double nrm = sqrt(2.0 / (double)D);
#pragma omp parallel for schedule(dynamic, 1)
  for (int M = 0; M < n_mol; ++M) {
    double* z = Z + (size_t)M * D;
    for (int l = 0; l < D; ++l) z[l] = 0.0;
    for (int64_t a = mol_off[M]; a < mol_off[M + 1]; ++a) {
      const int e = elem[a];
      for (int l = 0; l < D; ++l) {
        const float* w = W + ((size_t)e * D + l) * d;
        double u = 0.0;
        for (int k = 0; k < d; ++k) u += (double)w[k] * (double)x[a * d + k];
        z[l] += nrm * cos(u + (double)bias[(size_t)e * D + l]);
      }
    }
  }
}
