/* qmll.h -- C-ABI of the B200 (sm_100a) SORF hot path of QML-Lightning (arXiv 2206.01580).
 *
 * Citations are /root/reference/PAPER.md line numbers + equation; "A<n>" are the readings of
 * DESIGN.md (section "Readings of the paper").
 *
 * Conventions for every call
 *   - ALL data pointers are DEVICE pointers (cudaMalloc'ed / torch CUDA tensors), caller-owned,
 *     row-major, densely packed, naturally aligned to 16 bytes.  The two parameter structs
 *     themselves (qmll_sorf_params, qmll_grad) live in HOST memory.
 *   - The library allocates nothing persistent and keeps no state between calls; scratch comes from
 *     `workspace` (device memory, 256-byte aligned, size from qmll_workspace_bytes()).
 *   - Calls enqueue work on `cuda_stream` (a cudaStream_t cast to void*, NULL = default stream) and
 *     return without synchronising; outputs are valid once the stream has been synchronised.
 *   - Return value: QMLL_OK (0) or a negative qmll_status.  No exceptions cross the boundary.  Only
 *     host-visible arguments are checked; device-side contents that break the documented contract
 *     (elem[i] >= n_elem, non-monotone mol_off, signs other than +1/-1, nbr_idx >= n_atoms) are
 *     undefined behaviour.
 *   - There is no CPU fallback: on a machine without an sm_100 device every compute call returns
 *     QMLL_ERR_UNSUPPORTED / QMLL_ERR_CUDA.
 *
 * Notation: n_atoms atoms in n_mol molecules (atoms of a molecule contiguous),
 * descriptor length d (power of two), D = N_F features = n_s stacks of d, T = N_transform,
 * S[e,s,t,:] the Rademacher diagonal D_{t+1} of element e and stack s, H the unnormalised
 * Sylvester-Walsh-Hadamard matrix in natural order (L163-165), c = sqrt(d)/sigma * d^(-T/2) (A2).
 */
#ifndef QMLL_H_
#define QMLL_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  QMLL_OK = 0,
  QMLL_ERR_INVALID_ARG = -1, /* null pointer, d not a power of two, D % d != 0, T not in 1..3, sigma <= 0,
                                negative sizes, bad gradient layout                                         */
  QMLL_ERR_UNSUPPORTED = -2, /* d outside 16..1024 (see qmll_sorf_params), device is not sm_100             */
  QMLL_ERR_WORKSPACE = -3,   /* workspace NULL / too small / misaligned                                      */
  QMLL_ERR_CUDA = -4         /* a CUDA runtime / driver call or a kernel launch failed                       */
} qmll_status;

/* The SORF "model" minus alpha (eq. 20, eq. 14; A1-A7). */
typedef struct {
  int32_t d;           /* descriptor length: power of two, supported 16, 32, 64, 128, 256, 512, 1024          */
  int32_t D;           /* number of features N_F, a positive multiple of d                                    */
  int32_t n_transform; /* T in {1, 2, 3}                                                                       */
  int32_t n_elem;      /* number of element classes E >= 1                                                     */
  float sigma;         /* kernel width > 0                                                                     */
  const int8_t* signs; /* device [E, D/d, T, d], entries +1 / -1; t = 0 is D_1 and multiplies x (A4)          */
  const float* bias;   /* device [E, D], b in [0, 2 pi] (eq. 14); per element (A6)                            */
} qmll_sorf_params;

enum { QMLL_GRAD_NONE = 0, QMLL_GRAD_DENSE = 1, QMLL_GRAD_NEIGHBOR = 2 };

/* Descriptor gradient d x_I[m] / d r_{j,k} in one of two layouts (A12, A13). */
typedef struct {
  int32_t layout;           /* QMLL_GRAD_DENSE or QMLL_GRAD_NEIGHBOR                                          */
  const float* dense;       /* DENSE: molecules concatenated; molecule M with n atoms holds [n, d, n, 3] =     */
                            /*        (I, m, j, k), I and j local atom indices                                 */
  const int64_t* dense_off; /* DENSE: device [n_mol + 1] offsets (in floats) of each molecule's block,        */
                            /*        dense_off[M+1] - dense_off[M] = 3 d n_M^2                                */
  const int32_t* nbr_idx;   /* NEIGHBOR: device [n_atoms, K]: global atom index j, or -1 = padding            */
  const float* nbr_val;     /* NEIGHBOR: device [n_atoms, K, d, 3] = d x_I[m] / d r_{j,k}, j = nbr_idx[I, q];  */
                            /*        self and duplicate j are legal and ACCUMULATE                            */
  int32_t K;                /* NEIGHBOR: neighbours per atom                                                    */
  int64_t dense_floats;     /* DENSE: total number of floats in `dense` (= dense_off[n_mol]); the host needs it to */
                            /*        size the workspace copy made by qmll_sorf_forward (columns made contiguous)  */
} qmll_grad;

/* Steps a1-a3 (+a7): Z[M, l] = sum_{I in M} sqrt(2/D) cos((W_{e_I} x_I)[l] + b[e_I, l])
 * (eq. 20, eq. 14, eq. 15), l = s*d + m (A5).
 * If `grad` and `G` are given also the force rows (derivative features, L137; sign A8)
 *   G[3*j + k, l] = -dZ[M(j), l] / d r_{j,k} = sum_I sqrt(2/D) sin(u_I[l] + b[e_I, l]) (W_{e_I} dx_I[:, j, k])[l]
 * so that [Z; G] alpha = [E; F].  Rows of G are ordered by global atom index j then k = x, y, z.
 *   x        [n_atoms, d] fp32          elem  [n_atoms] int32 in [0, n_elem)
 *   mol_off  [n_mol + 1] int32, mol_off[0] = 0, mol_off[n_mol] = n_atoms, non-decreasing (empty molecules legal)
 *   Z        [n_mol, D] fp32, overwritten (may be NULL if only G is wanted)
 *   G        [3 n_atoms, D] fp32, overwritten; NULL unless grad != NULL
 * n_atoms == 0 or n_mol == 0 is legal (Z rows of empty molecules are zero). */
int qmll_sorf_forward(const qmll_sorf_params* p, const float* x, const int32_t* elem, const int32_t* mol_off,
                      int64_t n_atoms, int32_t n_mol, const qmll_grad* grad, float* Z, float* G,
                      void* workspace, size_t workspace_bytes, void* cuda_stream);

/* The same call with an explicit choice of how the force rows of a DENSE gradient are computed (both give the same
 * linear map applied to the same inputs, to fp32 accuracy):
 *   QMLL_ROWS_FWHT  every gradient column goes through the register Walsh-Hadamard / sign chain (any d).
 *   QMLL_ROWS_MMA   the chain of each (element, stack) is expanded once into its d x d integer matrix (exact in
 *                   fp16 for d <= 256) and applied to the columns on the tensor cores (tcgen05, columns split into
 *                   fp16 hi + lo); d = 128 or 256 only, else QMLL_ERR_UNSUPPORTED.
 *   QMLL_ROWS_MMA2  the same product on CTA pairs (tcgen05 cta_group::2: an MMA spans two SMs, each holds its own stacks'
 *                   W and half of the gradient columns); same support as QMLL_ROWS_MMA.
 *   QMLL_ROWS_AUTO  MMA2 where supported, else FWHT (what qmll_sorf_forward does). */
enum { QMLL_ROWS_AUTO = 0, QMLL_ROWS_FWHT = 1, QMLL_ROWS_MMA = 2, QMLL_ROWS_MMA2 = 3 };
int qmll_sorf_forward_mode(const qmll_sorf_params* p, const float* x, const int32_t* elem, const int32_t* mol_off,
                           int64_t n_atoms, int32_t n_mol, const qmll_grad* grad, float* Z, float* G,
                           void* workspace, size_t workspace_bytes, int32_t force_rows_mode, void* cuda_stream);

/* Steps a1, a5, a6: F[j, k] = -dE/dr_{j,k} with E = sum_M Z[M, :] . alpha  (eq. 15; F = -dE/dr,
 * eq. 5/10 L63, L90): q[l] = -sqrt(2/D) alpha[l] sin(u_I[l] + b); g_I = sum_s W_{e,s}^T q_s (transposed
 * Hadamard / sign chain, L268 "backwards pass"); F[j,k] = -sum_I sum_m g_I[m] dx_I[m]/dr_{j,k}.
 *   alpha [D] fp32;  grad required;  forces [n_atoms, 3] fp32, overwritten. */
int qmll_sorf_backward_forces(const qmll_sorf_params* p, const float* x, const int32_t* elem,
                              const int32_t* mol_off, int64_t n_atoms, int32_t n_mol, const float* alpha,
                              const qmll_grad* grad, float* forces, void* workspace, size_t workspace_bytes,
                              void* cuda_stream);

/* Step a8: normal equations (eq. 16, eq. 17; FP32 round-off remark L351):
 *   ZtZ (+)= A^T A,  Zty (+)= A^T y   for a block of rows A [rows, D] fp32 (rows of Z and/or G), y [rows] fp32.
 * ZtZ [D, D] fp32 is stored full and exactly symmetric; Zty [D] fp32 (summed in fp64, deterministic).
 * accumulate = 0 overwrites, 1 adds to the existing (symmetric) content.  The product runs on the tensor cores
 * with every operand split into hi + lo parts of 11 significant bits each (hi*hi + hi*lo + lo*hi, fp32
 * accumulate) and the row dimension cut into 128-row chunks that are summed in fp32 round-to-nearest.
 * lambda*I and the solve are the caller's (A10).  rows == 0 is legal (accumulate = 0 then zeroes the outputs).
 * y and Zty may both be NULL (ZtZ only).  Any D >= 1 is supported.
 * qmll_normal_equations uses QMLL_NE_SPLIT_F16; qmll_normal_equations_mode selects the operand container:
 *   QMLL_NE_SPLIT_F16   hi/lo in fp16 (same 11 significant bits as TF32, twice the MMA rate, half the bytes); one
 *                       power-of-two scale per (128-row chunk, 128-column block) keeps the parts inside fp16's
 *                       exponent range and is undone exactly.  Entries smaller than 2^-38 of the largest entry of
 *                       their 128 x 128 block lose their low bits (irrelevant for the Frobenius-norm accuracy of
 *                       a Gram matrix; use QMLL_NE_SPLIT_TF32 if single tiny entries matter).
 *   QMLL_NE_SPLIT_TF32  hi/lo in TF32 (the 3xTF32 scheme): full fp32 exponent range, half the speed.
 *   QMLL_NE_SPLIT_F16_PAIRS  the arithmetic of QMLL_NE_SPLIT_F16, bit for bit, on CTA pairs (tcgen05 cta_group::2: a
 *                       256 x 256 block of ZtZ per pair of SMs, each SM loads its own 128 rows of one operand and half
 *                       of the other).  Same workspace.  Measured: 3 % faster at D = 8192, 9 % slower at D = 16384 (the
 *                       kernel runs under the power cap either way), so it is not the default. */
enum { QMLL_NE_SPLIT_F16 = 0, QMLL_NE_SPLIT_TF32 = 1, QMLL_NE_SPLIT_F16_PAIRS = 2 };
int qmll_normal_equations(const float* A, const float* y, int64_t rows, int32_t D, int32_t accumulate,
                          float* ZtZ, float* Zty, void* workspace, size_t workspace_bytes, void* cuda_stream);
int qmll_normal_equations_mode(const float* A, const float* y, int64_t rows, int32_t D, int32_t accumulate,
                               float* ZtZ, float* Zty, void* workspace, size_t workspace_bytes, int32_t mode,
                               void* cuda_stream);

/* NEXT row f2: the per-element PCA projection that produces the SORF input from the raw
 * representation (eq. 21-22; "each element ... has its own projection matrix", L264):
 *   x[I, m] = sum_k rho[I, k] U[e_I, k, m]                      rho_I^T U_e^{N_PCA},  N_PCA = d
 * and, if grad_out != NULL, the same projection of a dense descriptor gradient (U is constant):
 *   grad_out (I, m, j, c) = sum_k grad_in (I, k, j, c) U[e_I, k, m]
 *   rho      [n_atoms, rep] fp32 (may be NULL if x is NULL)      elem [n_atoms] int32 in [0, n_elem)
 *   U        [n_elem, rep, d] fp32: the first d columns of every element's U_e (eq. 21); d a multiple of 4
 *   x        [n_atoms, d] fp32 out (may be NULL)
 *   grad_in  dense layout A12 with rep as the descriptor length: molecule M (n atoms) holds [n, rep, n, 3] at float
 *            offset grad_in_off[M]; grad_out holds [n, d, n, 3] at grad_out_off[M] (= the `dense` / `dense_off` of
 *            qmll_grad); mol_off as in qmll_sorf_forward (needed only with a gradient).
 * Plain fp32 FMAs (accuracy of an fp32 dot product of length rep); no workspace. */
int qmll_project(const float* rho, const int32_t* elem, const int32_t* mol_off, int64_t n_atoms, int32_t n_mol,
                 int32_t rep, int32_t d, int32_t n_elem, const float* U, float* x, const float* grad_in,
                 const int64_t* grad_in_off, float* grad_out, const int64_t* grad_out_off, void* cuda_stream);

/* NEXT row f3: the FCHL19 atomic representation (section E, eq. 23-33;
 * Table I) and its Jacobian with respect to the atomic positions, which make the path start from
 * coordinates: qmll_fchl19 -> qmll_project / qmll_project_neighbor -> qmll_sorf_forward / qmll_predict.
 *   two-body  (eq. 24-27): rho_i[X, s] = sum_{j: Z_j = X} f_cut(r_ij) r_ij^-N2 LogNormal(R_s; mu(r_ij), sigma(r_ij))
 *   three-body (eq. 28-33): rho_i[{X,Y}, s, a] = sum_{j<k, {Z_j, Z_k} = {X, Y}} xi_3 G_radial,s G_angular,a
 *                                                 f_cut(r_ij) f_cut(r_ik) f_cut(r_jk),  a = cos, sin (n = 1)
 * Readings (B1-B9): R_s = r_cut (s + 1) / n; f_cut = 0 beyond r_cut; unordered neighbour pairs; layout of
 * rho_i = [X][s] for X < n_elem, then [pair p(X <= Y) = X E - X (X - 1) / 2 + (Y - X)][s][cos, sin]:
 *   rep = n_elem n2 + n_elem (n_elem + 1) n3. */
typedef struct {
  int32_t n_elem;          /* element classes E, 1..16                                                         */
  int32_t n2, n3;          /* radial grid points of the two- and three-body terms, 1..32 (Table I: 23/24, 22/20) */
  float eta2, eta3;        /* widths (eq. 25-26, eq. 29)                                                       */
  float two_body_decay;    /* N_2 (eq. 24)                                                                     */
  float three_body_decay;  /* N_3 (eq. 30)                                                                     */
  float three_body_weight; /* c_3 (eq. 30)                                                                     */
  float zeta;              /* angular width (eq. 32-33); Table I: pi                                           */
  float r_cut;             /* cut-off radius > 0 (eq. 27); Table I: 6.0                                        */
} qmll_fchl19_params;

#define QMLL_FCHL19_MAX_NEIGHBOURS 160 /* neighbours INSIDE r_cut per atom the kernel holds on chip */

/* Length of rho_i for these parameters (host arithmetic). */
int32_t qmll_fchl19_rep_size(const qmll_fchl19_params* fp);

/*   r        [n_atoms, 3] fp32 positions;  elem [n_atoms] int32 in [0, n_elem)
 *   nbr_idx  [n_atoms, K] int32: candidate neighbours of atom i (global index j, -1 = padding); slot q stands for the
 *            image r[j] + nbr_shift[i, q, :] (nbr_shift [n_atoms, K, 3] fp32, NULL = no shifts: isolated molecules).
 *            The list is the caller's (neighbour search / periodic images are not part of this library); entries at
 *            or beyond r_cut contribute nothing; an atom must not list itself with a zero shift.
 *   rho      [n_atoms, rep] fp32 out
 *   jac_idx  [n_atoms, K + 1] int32 out, jac_val [n_atoms, K + 1, rep, 3] fp32 out, both NULL = representation only:
 *            slot 0 is the atom itself (jac_idx = i), slot 1 + q the image of neighbour slot q (jac_idx = j, or -1 and
 *            a zero block if that slot is padding or outside r_cut);
 *            jac_val[i, slot, k, c] = d rho_i[k] / d (position of that slot's atom)_c.  This is the NEIGHBOR layout of
 *            qmll_grad with descriptor length rep and K + 1 neighbours (images are independent variables; qmll_predict
 *            adds their contributions into the force on atom j).
 *   info     device int32 out: 0, or 1 + index of an atom with more than QMLL_FCHL19_MAX_NEIGHBOURS neighbours inside
 *            r_cut (its result is then incomplete).
 * Collinear triplets (sin theta = 0) have an unbounded d sin theta / d r; the kernel clamps sin theta at 1e-6 there.
 * fp32 arithmetic; no workspace. */
int qmll_fchl19(const qmll_fchl19_params* fp, const float* r, const int32_t* elem, int64_t n_atoms,
                const int32_t* nbr_idx, const float* nbr_shift, int32_t K, float* rho, int32_t* jac_idx,
                float* jac_val, int32_t* info, void* cuda_stream);

/* The backward pass of the same chain WITHOUT a Jacobian (what the paper does for prediction, L268: "for the backwards
 * pass ... the force components are stored and summed in on-chip memory"):
 *   coordinates -> qmll_fchl19 -> qmll_project -> qmll_sorf_backward_g -> qmll_project_back -> qmll_fchl19_backward.
 *
 * qmll_sorf_backward_g: g[I, m] = dE / dx_I[m] = -c sum_s (W_{e,s}^T (sqrt(2/D) alpha .* sin(u_I + b)))[m]  (step a5 alone,
 *   [n_atoms, d] fp32 out) and, if energies != NULL, the energies of qmll_predict.  Workspace as QMLL_CALL_PREDICT.
 * qmll_project_back:    w[I, k] = sum_m U[e_I, k, m] g[I, m] = dE / d rho_I[k]     ([n_atoms, rep] fp32 out).
 * qmll_fchl19_backward: forces[j, c] = -sum_I sum_k w[I, k] d rho_I[k] / d r_{j,c}  ([n_atoms, 3] fp32, overwritten); the
 *   sum runs over every atom I and every neighbour image of I (contributions of an image are added to the atom it is an
 *   image of) plus I itself.  Arguments as qmll_fchl19. */
int qmll_sorf_backward_g(const qmll_sorf_params* p, const float* x, const int32_t* elem, const int32_t* mol_off,
                         int64_t n_atoms, int32_t n_mol, const float* alpha, float* energies, float* g,
                         void* workspace, size_t workspace_bytes, void* cuda_stream);
int qmll_project_back(const float* g, const int32_t* elem, int64_t n_atoms, int32_t rep, int32_t d, int32_t n_elem,
                      const float* U, float* w, void* cuda_stream);
int qmll_fchl19_backward(const qmll_fchl19_params* fp, const float* r, const int32_t* elem, int64_t n_atoms,
                         const int32_t* nbr_idx, const float* nbr_shift, int32_t K, const float* w, float* forces,
                         int32_t* info, void* cuda_stream);

/* The per-element projection (qmll_project) of a NEIGHBOR-layout gradient, e.g. the Jacobian of qmll_fchl19:
 *   grad_out[I, q, m, c] = sum_k grad_in[I, q, k, c] U[e_I, k, m]
 *   grad_in [n_atoms, S, rep, 3] fp32, grad_out [n_atoms, S, d, 3] fp32, U [n_elem, rep, d] fp32, d % 4 == 0.
 * idx [n_atoms, S] int32 (may be NULL): blocks whose idx is negative are not read and are written as zeros. */
int qmll_project_neighbor(const float* grad_in, const int32_t* idx, const int32_t* elem, int64_t n_atoms, int32_t S,
                          int32_t rep, int32_t d, int32_t n_elem, const float* U, float* grad_out,
                          void* cuda_stream);

/* NEXT row f4 (variants): the feature map of steps a1-a3 on the TENSOR CORES.
 *
 * qmll_sorf_forward_mma: the same Z as qmll_sorf_forward(grad = NULL).  The chain of every (element, stack) is expanded
 *   once into its d x d integer matrix (exact in fp16 for d <= 256), atoms are sorted by element, x is split into fp16
 *   hi + lo, and U = W X runs on tcgen05 with the cos and the per-molecule sum in the epilogue (fp32 reductions into Z:
 *   the summation order over the atoms of a molecule is not fixed, results agree to fp32 rounding).  d = 128 or 256 and
 *   n_elem <= 16, else QMLL_ERR_UNSUPPORTED.  Workspace: qmll_featmap_workspace_bytes(d, D, n_elem, n_atoms, 0).
 *
 * qmll_rff_forward: the random Fourier feature map with a DENSE matrix (eq. 12-14, 18 L99-121, L150-152; the paper's
 *   RFF-versus-SORF comparison, Fig. 1):
 *     Z[M, l] = sum_{I in M} sqrt(2/D) cos( sum_k W[e_I, l, k] x_I[k] + b[e_I, l] )
 *   W [n_elem, D, d] fp32 (row l = w_l, the 1/sigma of eq. 18 already applied), bias [n_elem, D] fp32; W and x are split
 *   into fp16 hi + lo (hi*hi + hi*lo + lo*hi, fp32 accumulate: fp32-level accuracy).  d = 128 or 256, D a multiple of
 *   4, n_elem <= 16.  Workspace: qmll_featmap_workspace_bytes(d, D, n_elem, n_atoms, 1). */
int qmll_sorf_forward_mma(const qmll_sorf_params* p, const float* x, const int32_t* elem, const int32_t* mol_off,
                          int64_t n_atoms, int32_t n_mol, float* Z, void* workspace, size_t workspace_bytes,
                          void* cuda_stream);
int qmll_rff_forward(const float* W, const float* bias, int32_t d, int32_t D, int32_t n_elem, const float* x,
                     const int32_t* elem, const int32_t* mol_off, int64_t n_atoms, int32_t n_mol, float* Z,
                     void* workspace, size_t workspace_bytes, void* cuda_stream);
size_t qmll_featmap_workspace_bytes(int32_t d, int32_t D, int32_t n_elem, int64_t n_atoms, int32_t rff);

/* Exchange step of data-parallel training: the normal equations are sums over rows, so
 * ranks that own different molecules add their ZtZ / Zty.  ZtZ is symmetric: pack its lower triangle row by row
 * (row i holds i + 1 entries at offset i (i + 1) / 2; D (D + 1) / 2 floats), all-reduce the packed buffer, unpack
 * (writes both triangles: exactly symmetric).  D <= 65535. */
int qmll_pack_lower(const float* ZtZ, int32_t D, float* packed, void* cuda_stream);
int qmll_unpack_lower(const float* packed, int32_t D, float* ZtZ, void* cuda_stream);

/* Steps a1-a6 composed: energies[M] = Z[M, :] . alpha (eq. 15) and, if grad != NULL, forces as in
 * qmll_sorf_backward_forces, from one pass that shares u between cos and sin; Z is never materialised.
 *   energies [n_mol] fp32, overwritten;  forces [n_atoms, 3] fp32 or NULL (then grad must be NULL). */
int qmll_predict(const qmll_sorf_params* p, const float* x, const int32_t* elem, const int32_t* mol_off,
                 int64_t n_atoms, int32_t n_mol, const float* alpha, const qmll_grad* grad, float* energies,
                 float* forces, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Step a4 alone: energies[M] = sum_l Z[M, l] alpha[l] (eq. 15) for a caller that already holds Z -- the
 * training matrix, or the output of qmll_sorf_forward_mma / qmll_rff_forward: the tensor-core feature map followed by
 * this call is the energies-only prediction of the f4 variants (config 3: 21.5 ms against 30.5 ms for qmll_predict).
 *   Z [n_mol, D] fp32 row-major (read once, streaming), alpha [D] fp32, energies [n_mol] fp32 overwritten.
 *   fp32 products, partial sums of D / 128 terms in fp32, combined in FP64.  No workspace.  n_mol = 0 is a no-op. */
int qmll_energies(const float* Z, const float* alpha, int64_t n_mol, int32_t D, float* energies, void* cuda_stream);

/* qmll_predict for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same operation, same arguments and same kernels as qmll_predict (steps a1, a4-a6:
 * eq. 14-15, forces L137 / eq. 17), but without the workspace arguments.  The scratch -- the model's
 * lane-permuted tables and the FP64 energy accumulators -- is a static device array of QMLL_PREDICT_STATIC_MAX_BYTES
 * inside the library, held by every GPU that loads the library until the process exits.  The call allocates nothing
 * (no cudaMalloc / cudaFree, no allocating library routine); the first call on a device looks up the array's device
 * address (cudaGetSymbolAddress), later calls reuse it.
 *   Limit: qmll_workspace_bytes(QMLL_CALL_PREDICT, p, n_atoms, n_mol, 0) <= qmll_predict_static_max_bytes(), else
 *   QMLL_ERR_WORKSPACE and nothing is launched (4 MiB covers D = 65536 with 5 elements and ~300 000 molecules per
 *   call; all five BASELINE configs fit).  Other errors as qmll_predict.
 *   Sharing: every call on a device uses the same array.  What must start at zero is cleared inside every call and
 *   the tables are rewritten in full, so back-to-back calls on one stream (or otherwise ordered) are independent;
 *   calls that OVERLAP on the GPU (different streams without ordering, concurrent graph launches) race on the
 *   scratch and give undefined results.  Thread-safe at enqueue. */
#define QMLL_PREDICT_STATIC_MAX_BYTES (4u << 20)
int qmll_predict_static(const qmll_sorf_params* p, const float* x, const int32_t* elem, const int32_t* mol_off,
                        int64_t n_atoms, int32_t n_mol, const float* alpha, const qmll_grad* grad, float* energies,
                        float* forces, void* cuda_stream);
size_t qmll_predict_static_max_bytes(void);

/* NEXT step after the accumulation: alpha = (ZtZ + lambda I)^-1 Zty, the regularised
 * normal equations of eq. 16-17 (L134-144; "solved by LU decomposition", L137 -- SPD, so a blocked Cholesky), in FP64.
 *   ZtZ [D, D] fp32 symmetric (only the lower triangle is read), Zty [D] fp32, lambda >= 0, alpha [D] fp32 out,
 *   info: device int32, LAPACK convention: 0 = success, k > 0 = leading minor of order k not positive definite
 *   (alpha is then NaN-contaminated).  The inputs are not modified.  D <= 65534 (else QMLL_ERR_UNSUPPORTED).
 *   Stream behaviour: panel factorisations run on an internal high-priority stream, forked from and joined back into
 *   `cuda_stream` with events (look-ahead, overlapping the trailing update); every effect of the call is ordered on
 *   `cuda_stream` as usual, and the pattern is stream-capturable.  The internal stream and its events are created
 *   once per device on first use and live for the process; concurrent calls are serialised at enqueue by a mutex. */
int qmll_solve(const float* ZtZ, const float* Zty, int32_t D, double lambda, float* alpha, int32_t* info,
               void* workspace, size_t workspace_bytes, void* cuda_stream);

enum {
  QMLL_CALL_FORWARD = 0,         /* qmll_sorf_forward without grad            */
  QMLL_CALL_FORWARD_GRAD = 1,    /* qmll_sorf_forward with grad and G         */
  QMLL_CALL_BACKWARD_FORCES = 2, /* qmll_sorf_backward_forces                 */
  QMLL_CALL_NORMAL_EQUATIONS = 3,/* qmll_normal_equations (uses rows and p->D; p->d may be 0) */
  QMLL_CALL_PREDICT = 4,         /* qmll_predict                              */
  QMLL_CALL_SOLVE = 5            /* qmll_solve (uses p->D only)               */
};

/* Scratch bytes the named call needs for these sizes (host-side arithmetic only, no CUDA call).
 * For QMLL_CALL_FORWARD_GRAD with a dense gradient pass rows = grad->dense_floats (0 for a neighbour gradient).
 * For QMLL_CALL_NORMAL_EQUATIONS this is the size that lets all `rows` be staged in one panel; the call
 * also runs (in several panels) with any workspace of at least qmll_normal_equations_min_workspace(D). */
size_t qmll_workspace_bytes(int which_call, const qmll_sorf_params* p, int64_t n_atoms, int32_t n_mol,
                            int64_t rows);
size_t qmll_normal_equations_min_workspace(int32_t D);
/* The same two sizes for an explicit mode (qmll_workspace_bytes / _min_workspace answer for QMLL_NE_SPLIT_F16). */
size_t qmll_normal_equations_workspace(int64_t rows, int32_t D, int32_t mode);
size_t qmll_normal_equations_min_workspace_mode(int32_t D, int32_t mode);

/* Static description of a status code; for QMLL_ERR_CUDA the text of the last CUDA error seen by this
 * thread is appended.  The returned pointer stays valid until the next call from the same thread. */
const char* qmll_status_string(int status);

#ifdef __cplusplus
}
#endif
#endif /* QMLL_H_ */
