/* oracle/fchl19_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, FP64 CPU statement of the FCHL19 atomic representation (arXiv 2206.01580, PAPER.md section E,
 * eqs. 23-33) and of its Jacobian with respect to the atomic positions.  It
 * shares no code, header, table or helper with the CUDA path and neither side includes the other.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * The representation is written ONCE, over complex coordinates, term by term as the paper prints it (vectors,
 * dot products, the three angles of the triangle).  The value is the function at real coordinates.  The Jacobian is
 * the complex-step derivative of the SAME function, d rho / d t = Im rho(t + i h) / h with h = 1e-30: no second set
 * of formulas that could be wrong independently, and no subtractive cancellation (exact to rounding for analytic
 * functions; every function used -- sqrt, log, exp, cos, powers with real exponents -- is analytic where it is
 * evaluated; the cut-off tests use the real parts).
 *
 * Inputs are the fp32 / int32 arrays the GPU library receives, widened to double.  Outputs are double.
 *
 * Readings of the paper where it is silent or garbled (DESIGN.md "Readings" B1-B9):
 *   B1 radial grids: R_s = r_cut (s + 1) / n, s = 0..n-1, for both the two-body (n = n_2) and the three-body
 *      (n = n_3) terms ("linearly distributed between 0 and r_cut", L190; R_s = 0 is excluded because eq. 24 needs
 *      ln R_s and divides by R_s).
 *   B2 f_cut(r) = 0 for r >= r_cut (eq. 27 only gives the inner branch; "smoothly decay ... to zero at r_cut").
 *   B3 eq. 28 multiplies THREE cut-offs, f(r_ij) f(r_jk) f(r_ik): taken as printed, so a triplet whose j-k distance
 *      is >= r_cut contributes nothing.
 *   B4 eq. 30's denominator "(r_ik r_jk r_ki)^N3" is the product of the three distinct side lengths.
 *   B5 eq. 31-33 (garbled): G^cos_n = exp(-(zeta n)^2 / 2) (cos(n theta) - cos(n (theta + pi))),
 *      G^sin_n = exp(-(zeta n)^2 / 2) (sin(n theta) - sin(n (theta + pi))), only n = 1 (L230): 2 exp(-zeta^2/2) cos
 *      theta and 2 exp(-zeta^2/2) sin theta, theta = theta_kij the angle at the central atom i, sin theta >= 0.
 *   B6 the three-body sum runs over UNORDERED pairs {j, k} of neighbours (each triangle once).
 *   B7 layout of rho_i: [two-body: element X = 0..E-1][s = 0..n_2-1], then [three-body: element pair p(X, Y),
 *      X <= Y, p = X E - X (X - 1) / 2 + (Y - X)][s = 0..n_3-1][cos, sin]; length E n_2 + E (E + 1) n_3.
 *      "For every unique combination of two elements X, Y" (eq. 23): the two-body block of an element is
 *      stored once, not once per pair.
 *   B8 neighbours are given as a list: slot q of atom i is the image r[nbr_idx[i, q]] + nbr_shift[i, q, :] (shift
 *      NULL = 0; -1 = padding); the list is the caller's (neighbour lists / periodic images are out of scope,
 *      L268 "simple tiled neighbour-list").  An atom must not list itself with zero shift.
 *   B9 Jacobian layout: slot 0 is the central atom i itself, slot 1 + q the image in neighbour slot q:
 *      jac[i, slot, k, c] = d rho_i[k] / d (position of that slot's atom)_c.  Images are independent variables.
 *
 * Pins (tests/test_fchl19_pins.py): the two-body term against scipy.stats.lognorm.pdf and the moments the paper's
 * mu, sigma are built to have (mean r_ij, variance eta_2); radial normalisation and centre of the three-body
 * Gaussian; closed forms for the equilateral and the right-angled triangle; rotation / translation / neighbour
 * order / element relabelling invariances; cut-off; additivity over pairs; the Jacobian against Richardson finite
 * differences, its translation sum rule and rotational consistency.  No function here is "parity unpinned".
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

typedef struct {
  int n_elem, n2, n3;
  double eta2, eta3, N2, N3, c3, zeta, rcut;
} fchl_par;

int qo_fchl19_rep_size(int n_elem, int n2, int n3) { return n_elem * n2 + n_elem * (n_elem + 1) * n3; }

static const double kPi = 3.14159265358979323846;

/* sqrt(v . v) for complex vectors: the analytic continuation of the Euclidean length (NOT the Hermitian norm) */
static cplx length3(const cplx* v) { return csqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]); }
static cplx dot3(const cplx* a, const cplx* b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
static cplx rpow(cplx r, double p) { return cexp(p * clog(r)); }       /* r^p, Re r > 0 */

/* eq. 27 (L201), inner branch; callers test Re r < r_cut (B2) */
static cplx f_cut(cplx r, double rcut) { return 0.5 * (ccos(kPi * r / rcut) + 1.0); }

/* rho_i as a function of the (complex) position of the central atom and of its neighbour images.
 *   centre[3], img[nn][3] positions, img_elem[nn] elements; out[rep] is overwritten. */
static void fchl19_atom(const fchl_par* P, const cplx* centre, const cplx (*img)[3], const int* img_elem, int nn,
                        cplx* out) {
  const int E = P->n_elem, rep = qo_fchl19_rep_size(E, P->n2, P->n3);
  for (int k = 0; k < rep; ++k) out[k] = 0.0;

  /* ---- two-body, eq. 24-27 (L186-201) ---- */
  for (int j = 0; j < nn; ++j) {
    cplx a[3] = {img[j][0] - centre[0], img[j][1] - centre[1], img[j][2] - centre[2]};
    const cplx r = length3(a);
    if (creal(r) >= P->rcut) continue;                                   /* B2 */
    const cplx sigma2 = clog(1.0 + P->eta2 / (r * r));                   /* eq. 26 */
    const cplx mu = clog(r / csqrt(1.0 + P->eta2 / (r * r)));            /* eq. 25 */
    const cplx sigma = csqrt(sigma2);
    for (int s = 0; s < P->n2; ++s) {
      const double Rs = P->rcut * (s + 1) / P->n2;                       /* B1 */
      const cplx t = log(Rs) - mu;
      out[img_elem[j] * P->n2 + s] += f_cut(r, P->rcut) * (1.0 / rpow(r, P->N2)) *
                                      (1.0 / (Rs * sigma * sqrt(2.0 * kPi))) * cexp(-(t * t) / (2.0 * sigma2));
    }
  }

  /* ---- three-body, eq. 28-33 (L203-230), unordered pairs (B6) ---- */
  const int off3 = E * P->n2;
  for (int j = 0; j < nn; ++j)
    for (int k = j + 1; k < nn; ++k) {
      cplx a[3], b[3], c[3], ma[3], mb[3], mc[3];
      for (int q = 0; q < 3; ++q) {
        a[q] = img[j][q] - centre[q];     /* i -> j */
        b[q] = img[k][q] - centre[q];     /* i -> k */
        c[q] = img[k][q] - img[j][q];     /* j -> k */
        ma[q] = -a[q]; mb[q] = -b[q]; mc[q] = -c[q];
      }
      const cplx rij = length3(a), rik = length3(b), rjk = length3(c);
      if (creal(rij) >= P->rcut || creal(rik) >= P->rcut || creal(rjk) >= P->rcut) continue;   /* B2, B3 */
      const cplx cos_i = dot3(a, b) / (rij * rik);      /* theta_kij: angle at i between j and k */
      const cplx cos_j = dot3(ma, c) / (rij * rjk);     /* theta_ijk: angle at j between i and k */
      const cplx cos_k = dot3(mb, mc) / (rik * rjk);    /* theta_jki: angle at k between i and j */
      const cplx theta = cacos(cos_i);                  /* theta_kij in [0, pi] */
      const cplx xi3 = P->c3 * (1.0 + 3.0 * cos_i * cos_j * cos_k) / rpow(rik * rjk * rij, P->N3);   /* eq. 30, B4 */
      const cplx cut = f_cut(rij, P->rcut) * f_cut(rjk, P->rcut) * f_cut(rik, P->rcut);               /* eq. 28 */
      const double n = 1.0;                                                                           /* L230 */
      const double damp = exp(-(P->zeta * n) * (P->zeta * n) / 2.0);
      const cplx g_cos = damp * (ccos(n * theta) - ccos(n * (theta + kPi)));                          /* eq. 32, B5 */
      const cplx g_sin = damp * (csin(n * theta) - csin(n * (theta + kPi)));                          /* eq. 33, B5 */
      int X = img_elem[j], Y = img_elem[k];
      if (X > Y) { int t = X; X = Y; Y = t; }
      const int p = X * E - X * (X - 1) / 2 + (Y - X);                                                /* B7 */
      for (int s = 0; s < P->n3; ++s) {
        const double Rs = P->rcut * (s + 1) / P->n3;                                                  /* B1 */
        const cplx m = 0.5 * (rij + rik) - Rs;
        const cplx radial = sqrt(P->eta3 / kPi) * cexp(-P->eta3 * m * m);                             /* eq. 29 */
        out[off3 + (p * P->n3 + s) * 2 + 0] += xi3 * radial * g_cos * cut;
        out[off3 + (p * P->n3 + s) * 2 + 1] += xi3 * radial * g_sin * cut;
      }
    }
}

/* gathers the images of atom i; returns their number, slot_of[m] = neighbour slot q of image m */
static int gather(const float* r, const int32_t* elem, const int32_t* nbr_idx, const float* nbr_shift, int K,
                  int64_t i, cplx (*img)[3], int* img_elem, int* slot_of) {
  int nn = 0;
  for (int q = 0; q < K; ++q) {
    const int32_t j = nbr_idx[i * K + q];
    if (j < 0) continue;
    for (int c = 0; c < 3; ++c)
      img[nn][c] = (double)r[3 * (int64_t)j + c] + (nbr_shift ? (double)nbr_shift[(i * K + q) * 3 + c] : 0.0);
    img_elem[nn] = elem[j];
    slot_of[nn] = q;
    ++nn;
  }
  return nn;
}

/* rho [n_atoms, rep] */
void qo_fchl19(const float* r, const int32_t* elem, int64_t n_atoms, const int32_t* nbr_idx, const float* nbr_shift,
               int K, int n_elem, int n2, int n3, double eta2, double eta3, double N2, double N3, double c3,
               double zeta, double rcut, double* rho) {
  const fchl_par P = {n_elem, n2, n3, eta2, eta3, N2, N3, c3, zeta, rcut};
  const int rep = qo_fchl19_rep_size(n_elem, n2, n3);
#pragma omp parallel
  {
    cplx (*img)[3] = malloc(sizeof(cplx[3]) * (K > 0 ? K : 1));
    int* img_elem = malloc(sizeof(int) * (K > 0 ? K : 1));
    int* slot_of = malloc(sizeof(int) * (K > 0 ? K : 1));
    cplx* out = malloc(sizeof(cplx) * (rep > 0 ? rep : 1));
#pragma omp for schedule(dynamic, 4)
    for (int64_t i = 0; i < n_atoms; ++i) {
      const int nn = gather(r, elem, nbr_idx, nbr_shift, K, i, img, img_elem, slot_of);
      cplx centre[3] = {r[3 * i], r[3 * i + 1], r[3 * i + 2]};
      fchl19_atom(&P, centre, (const cplx (*)[3])img, img_elem, nn, out);
      for (int k = 0; k < rep; ++k) rho[i * rep + k] = creal(out[k]);
    }
    free(img); free(img_elem); free(slot_of); free(out);
  }
}

/* Jacobian of the atoms listed in `atoms[n_sel]`: jac [n_sel, K + 1, rep, 3] (B9), complex-step derivative. */
void qo_fchl19_jacobian(const float* r, const int32_t* elem, const int32_t* nbr_idx, const float* nbr_shift, int K,
                        const int64_t* atoms, int64_t n_sel, int n_elem, int n2, int n3, double eta2, double eta3,
                        double N2, double N3, double c3, double zeta, double rcut, double* jac) {
  const fchl_par P = {n_elem, n2, n3, eta2, eta3, N2, N3, c3, zeta, rcut};
  const int rep = qo_fchl19_rep_size(n_elem, n2, n3);
  const double h = 1e-30;
  memset(jac, 0, sizeof(double) * (size_t)n_sel * (K + 1) * rep * 3);
#pragma omp parallel
  {
    cplx (*img)[3] = malloc(sizeof(cplx[3]) * (K > 0 ? K : 1));
    int* img_elem = malloc(sizeof(int) * (K > 0 ? K : 1));
    int* slot_of = malloc(sizeof(int) * (K > 0 ? K : 1));
    cplx* out = malloc(sizeof(cplx) * (rep > 0 ? rep : 1));
#pragma omp for schedule(dynamic, 1) collapse(2)
    for (int64_t t = 0; t < n_sel; ++t)
      for (int v = 0; v < 3 * (K + 1); ++v) {       /* v = (slot, coordinate) */
        const int64_t i = atoms[t];
        const int slot = v / 3, c = v % 3;
        const int nn = gather(r, elem, nbr_idx, nbr_shift, K, i, img, img_elem, slot_of);
        cplx centre[3] = {r[3 * i], r[3 * i + 1], r[3 * i + 2]};
        if (slot == 0) {
          centre[c] += h * I;
        } else {
          int m = -1;
          for (int q = 0; q < nn; ++q) if (slot_of[q] == slot - 1) m = q;
          if (m < 0) continue;                       /* padding slot: zero block */
          img[m][c] += h * I;
        }
        fchl19_atom(&P, centre, (const cplx (*)[3])img, img_elem, nn, out);
        double* dst = jac + ((size_t)t * (K + 1) + slot) * rep * 3;
        for (int k = 0; k < rep; ++k) dst[k * 3 + c] = cimag(out[k]) / h;
      }
    free(img); free(img_elem); free(slot_of); free(out);
  }
}

/* Per-element PCA projection of a neighbour-layout Jacobian (eq. 21-22; U is constant):
 *   out[at, slot, m, c] = sum_k in[at, slot, k, c] U[e_at, k, m].    in [n_atoms, S, rep, 3] fp32, out [n_atoms, S, d, 3] */
void qo_project_neighbor_gradient(const float* gin, const int32_t* elem, int64_t n_atoms, int S, int rep, int d,
                                  const float* U, double* gout) {
#pragma omp parallel for schedule(static)
  for (int64_t at = 0; at < n_atoms; ++at) {
    const float* Ue = U + (size_t)elem[at] * rep * d;
    for (int s = 0; s < S; ++s)
      for (int m = 0; m < d; ++m)
        for (int c = 0; c < 3; ++c) {
          double acc = 0.0;
          for (int k = 0; k < rep; ++k)
            acc += (double)gin[(((size_t)at * S + s) * rep + k) * 3 + c] * (double)Ue[(size_t)k * d + m];
          gout[(((size_t)at * S + s) * d + m) * 3 + c] = acc;
        }
  }
}

/* The same function for ONE atom given in double precision (for the pins: finite differences need FP64 positions).
 *   rho [rep];  jac [nn + 1, rep, 3] (slot 0 = centre, slot 1 + m = image m) or NULL. */
void qo_fchl19_atom_f64(const double* centre, const double* img /* [nn, 3] */, const int32_t* img_elem, int nn,
                        int n_elem, int n2, int n3, double eta2, double eta3, double N2, double N3, double c3,
                        double zeta, double rcut, double* rho, double* jac) {
  const fchl_par P = {n_elem, n2, n3, eta2, eta3, N2, N3, c3, zeta, rcut};
  const int rep = qo_fchl19_rep_size(n_elem, n2, n3);
  const double h = 1e-30;
  cplx (*z)[3] = malloc(sizeof(cplx[3]) * (nn > 0 ? nn : 1));
  int* ze = malloc(sizeof(int) * (nn > 0 ? nn : 1));
  cplx* out = malloc(sizeof(cplx) * (rep > 0 ? rep : 1));
  for (int v = -1; v < (jac ? 3 * (nn + 1) : 0); ++v) {
    cplx c0[3] = {centre[0], centre[1], centre[2]};
    for (int m = 0; m < nn; ++m) {
      for (int c = 0; c < 3; ++c) z[m][c] = img[3 * m + c];
      ze[m] = img_elem[m];
    }
    if (v >= 0) {
      if (v / 3 == 0) c0[v % 3] += h * I; else z[v / 3 - 1][v % 3] += h * I;
    }
    fchl19_atom(&P, c0, (const cplx (*)[3])z, ze, nn, out);
    if (v < 0) for (int k = 0; k < rep; ++k) rho[k] = creal(out[k]);
    else for (int k = 0; k < rep; ++k) jac[((size_t)(v / 3) * rep + k) * 3 + v % 3] = cimag(out[k]) / h;
  }
  free(z); free(ze); free(out);
}

/* Backward pass of the projection x = rho^T U_e (eq. 22): w[at, k] = dE/d rho[at, k] = sum_m U[e_at, k, m] g[at, m]. */
void qo_project_back(const double* g, const int32_t* elem, int64_t n_atoms, int rep, int d, const float* U, double* w) {
#pragma omp parallel for schedule(static)
  for (int64_t at = 0; at < n_atoms; ++at) {
    const float* Ue = U + (size_t)elem[at] * rep * d;
    for (int k = 0; k < rep; ++k) {
      double acc = 0.0;
      for (int m = 0; m < d; ++m) acc += (double)Ue[(size_t)k * d + m] * g[at * d + m];
      w[at * rep + k] = acc;
    }
  }
}

/* Backward pass of the representation: F[j, c] = -sum_i sum_k w[i, k] d rho_i[k] / d r_{j,c}, summed over every atom i,
 * the atom itself (slot 0 of its Jacobian) and its neighbour images (slot 1 + q -> atom nbr_idx[i, q]).  Plain
 * contraction of the complex-step Jacobian above (the definition), nothing fused. */
void qo_fchl19_backward(const float* r, const int32_t* elem, int64_t n_atoms, const int32_t* nbr_idx,
                        const float* nbr_shift, int K, const double* w, int n_elem, int n2, int n3, double eta2,
                        double eta3, double N2, double N3, double c3, double zeta, double rcut, double* F) {
  const int rep = qo_fchl19_rep_size(n_elem, n2, n3);
  for (int64_t t = 0; t < 3 * n_atoms; ++t) F[t] = 0.0;
  double* jac = malloc(sizeof(double) * (size_t)(K + 1) * rep * 3);
  for (int64_t i = 0; i < n_atoms; ++i) {
    qo_fchl19_jacobian(r, elem, nbr_idx, nbr_shift, K, &i, 1, n_elem, n2, n3, eta2, eta3, N2, N3, c3, zeta, rcut, jac);
    for (int slot = 0; slot <= K; ++slot) {
      const int64_t j = slot == 0 ? i : nbr_idx[i * K + slot - 1];
      if (j < 0) continue;
      for (int k = 0; k < rep; ++k)
        for (int c = 0; c < 3; ++c) F[3 * j + c] -= w[i * rep + k] * jac[((size_t)slot * rep + k) * 3 + c];
    }
  }
  free(jac);
}
