// qmll_api.cu -- the C-ABI of include/qmll.h: host-side argument checks, workspace carving and the
// sequencing of the kernels.  Every step of the path runs in the kernels; nothing is computed on the host.
#include <atomic>
#include <stdio.h>
#include <string.h>

#include "qmll_common.cuh"

namespace qmll {

static thread_local char g_err_text[512] = "";
static std::atomic<long long> g_launches{0};

void note_cuda_error(cudaError_t err, const char* where) {
  snprintf(g_err_text, sizeof(g_err_text), "%s: %s", where, cudaGetErrorString(err));
  cudaGetLastError();  // clear the sticky-less error state
}
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

static int check_params(const qmll_sorf_params* p) {
  if (!p || !p->signs || !p->bias) return QMLL_ERR_INVALID_ARG;
  if (p->d <= 0 || (p->d & (p->d - 1)) != 0) return QMLL_ERR_INVALID_ARG;
  if (p->D <= 0 || p->D % p->d != 0) return QMLL_ERR_INVALID_ARG;
  if (p->n_transform < 1 || p->n_transform > 3) return QMLL_ERR_INVALID_ARG;
  if (p->n_elem < 1 || !(p->sigma > 0.f)) return QMLL_ERR_INVALID_ARG;
  if (!sorf_supported_d(p->d)) return QMLL_ERR_UNSUPPORTED;
  return QMLL_OK;
}

static int check_problem(const float* x, const int32_t* elem, const int32_t* mol_off, int64_t n_atoms,
                         int32_t n_mol) {
  if (n_atoms < 0 || n_mol < 0 || n_atoms > 0x7fffff00LL) return QMLL_ERR_INVALID_ARG;
  if (!mol_off) return QMLL_ERR_INVALID_ARG;
  if (n_atoms > 0 && (!x || !elem || n_mol == 0)) return QMLL_ERR_INVALID_ARG;
  return QMLL_OK;
}

static int check_grad(const qmll_grad* g) {
  if (!g) return QMLL_ERR_INVALID_ARG;
  if (g->layout == QMLL_GRAD_DENSE)
    return (g->dense && g->dense_off && g->dense_floats >= 0) ? QMLL_OK : QMLL_ERR_INVALID_ARG;
  if (g->layout == QMLL_GRAD_NEIGHBOR) {
    if (g->K < 0) return QMLL_ERR_INVALID_ARG;
    return (g->K == 0 || (g->nbr_idx && g->nbr_val)) ? QMLL_OK : QMLL_ERR_INVALID_ARG;
  }
  return QMLL_ERR_INVALID_ARG;
}

static int check_device() {
  int dev = 0, major = 0, minor = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev);
  if (e != cudaSuccess) { note_cuda_error(e, "cudaGetDevice"); return QMLL_ERR_CUDA; }
  return (major == 10 && minor == 0) ? QMLL_OK : QMLL_ERR_UNSUPPORTED;  // the kernels are built for sm_100a only
}

static int check_ws(void* ws, size_t have, size_t need) {
  if (need == 0) return QMLL_OK;
  if (!ws || ((uintptr_t)ws & 255) != 0 || have < need) return QMLL_ERR_WORKSPACE;
  return QMLL_OK;
}

static size_t zs_bytes(const qmll_sorf_params* p, int64_t n_atoms) {
  return align_up(sorf_zs_floats(p, n_atoms) * sizeof(float), 256) + 256;
}
// scratch of the dense force-row step: the transposed gradient (FWHT path) or W table + split columns (tensor path)
static bool use_rows_mma(const qmll_sorf_params* p, int32_t mode) {
  return mode != QMLL_ROWS_FWHT && sorf_mma_supported(p);
}
static size_t rows_scratch_bytes(const qmll_sorf_params* p, int64_t n_atoms, int32_t n_mol, int64_t dense_floats,
                                 bool mma) {
  if (!mma) return align_up((size_t)(dense_floats > 0 ? dense_floats : 0) * 4, 256) + 256;
  return align_up(sorf_mma_w_bytes(p), 256) + 2 * align_up(sorf_mma_x_bytes(p, n_atoms, dense_floats), 256) +
         align_up(((size_t)n_mol + 1) * sizeof(long long), 256) + align_up((size_t)n_atoms * sizeof(float), 256) + 5 * 256;
}
static size_t e_bytes(int32_t n_mol) { return align_up((size_t)n_mol * sizeof(double), 256) + 256; }

// shared body of qmll_sorf_backward_forces and qmll_predict
static int backward_impl(const qmll_sorf_params* p, const float* x, const int32_t* elem, const int32_t* mol_off,
                         int64_t n_atoms, int32_t n_mol, const float* alpha, const qmll_grad* grad, float* energies,
                         float* forces, void* workspace, size_t workspace_bytes, cudaStream_t st, int which,
                         float* g_out = nullptr) {
  int rc = check_params(p);
  if (rc) return rc;
  rc = check_problem(x, elem, mol_off, n_atoms, n_mol);
  if (rc) return rc;
  if (!alpha) return QMLL_ERR_INVALID_ARG;
  if (forces) { rc = check_grad(grad); if (rc) return rc; }
  else if (grad) return QMLL_ERR_INVALID_ARG;
  if (!forces && !energies && !g_out) return QMLL_ERR_INVALID_ARG;
  if (g_out && forces) return QMLL_ERR_INVALID_ARG;
  rc = check_device();
  if (rc) return rc;
  rc = check_ws(workspace, workspace_bytes, qmll_workspace_bytes(which, p, n_atoms, n_mol, 0));
  if (rc) return rc;

  Carver ws(workspace, workspace_bytes);
  SorfTables t;
  rc = sorf_prepare_tables(p, alpha, ws, &t, st);
  if (rc) return rc;
  double* eacc = energies ? ws.take<double>((size_t)n_mol) : nullptr;
  if (!ws.fits()) return QMLL_ERR_WORKSPACE;
  if (eacc && n_mol > 0) QMLL_CUDA_TRY(cudaMemsetAsync(eacc, 0, (size_t)n_mol * sizeof(double), st));
  if (forces && n_atoms > 0) QMLL_CUDA_TRY(cudaMemsetAsync(forces, 0, (size_t)n_atoms * 3 * sizeof(float), st));
  SorfProblem pr{p, x, elem, mol_off, n_atoms, n_mol};
  rc = g_out ? sorf_launch_predict(pr, t, nullptr, g_out, eacc, st, true)
             : sorf_launch_predict(pr, t, forces ? grad : nullptr, forces, eacc, st);
  if (rc) return rc;
  if (energies) { rc = sorf_finish_energies(eacc, energies, n_mol, st); if (rc) return rc; }
  return QMLL_OK;
}

}  // namespace qmll

using namespace qmll;

extern "C" {

static bool valid_mode(int32_t mode) {
  return mode == QMLL_NE_SPLIT_F16 || mode == QMLL_NE_SPLIT_TF32 || mode == QMLL_NE_SPLIT_F16_PAIRS;
}
size_t qmll_normal_equations_min_workspace(int32_t D) { return D > 0 ? syrk_min_workspace(D, QMLL_NE_SPLIT_F16) : 0; }
size_t qmll_normal_equations_min_workspace_mode(int32_t D, int32_t mode) {
  return (D > 0 && valid_mode(mode)) ? syrk_min_workspace(D, mode) : 0;
}
size_t qmll_normal_equations_workspace(int64_t rows, int32_t D, int32_t mode) {
  return (D > 0 && valid_mode(mode)) ? syrk_full_workspace(rows, D, mode) : 0;
}

size_t qmll_workspace_bytes(int which_call, const qmll_sorf_params* p, int64_t n_atoms, int32_t n_mol,
                            int64_t rows) {
  if (!p) return 0;
  if (which_call == QMLL_CALL_NORMAL_EQUATIONS) return p->D > 0 ? syrk_full_workspace(rows, p->D, QMLL_NE_SPLIT_F16) : 0;
  if (which_call == QMLL_CALL_SOLVE) return p->D > 0 ? solve_workspace_bytes(p->D) : 0;
  if (p->d <= 0 || p->D <= 0 || p->D % p->d != 0 || p->n_elem < 1 || p->n_transform < 1 || !sorf_supported_d(p->d))
    return 0;
  if (n_atoms < 0) n_atoms = 0;
  if (n_mol < 0) n_mol = 0;
  switch (which_call) {
    case QMLL_CALL_FORWARD: return sorf_tables_bytes(p, false);
    case QMLL_CALL_FORWARD_GRAD: {   // enough for either force-row path
      const size_t a = rows_scratch_bytes(p, n_atoms, n_mol, rows, false);
      const size_t b = sorf_mma_supported(p) ? rows_scratch_bytes(p, n_atoms, n_mol, rows, true) : 0;
      return sorf_tables_bytes(p, false) + zs_bytes(p, n_atoms) + (a > b ? a : b);
    }
    case QMLL_CALL_BACKWARD_FORCES: return sorf_tables_bytes(p, true);
    case QMLL_CALL_PREDICT: return sorf_tables_bytes(p, true) + e_bytes(n_mol);
    default: return 0;
  }
}

int qmll_sorf_forward_mode(const qmll_sorf_params* p, const float* x, const int32_t* elem, const int32_t* mol_off,
                           int64_t n_atoms, int32_t n_mol, const qmll_grad* grad, float* Z, float* G, void* workspace,
                           size_t workspace_bytes, int32_t force_rows_mode, void* cuda_stream) {
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int rc = check_params(p);
  if (rc) return rc;
  rc = check_problem(x, elem, mol_off, n_atoms, n_mol);
  if (rc) return rc;
  if ((G != nullptr) != (grad != nullptr)) return QMLL_ERR_INVALID_ARG;
  if (!Z && !G) return QMLL_ERR_INVALID_ARG;
  if (force_rows_mode < QMLL_ROWS_AUTO || force_rows_mode > QMLL_ROWS_MMA2) return QMLL_ERR_INVALID_ARG;
  if (grad) { rc = check_grad(grad); if (rc) return rc; }
  if ((force_rows_mode == QMLL_ROWS_MMA || force_rows_mode == QMLL_ROWS_MMA2) && !(grad && grad->layout == QMLL_GRAD_DENSE && sorf_mma_supported(p)))
    return QMLL_ERR_UNSUPPORTED;
  rc = check_device();
  if (rc) return rc;
  rc = check_ws(workspace, workspace_bytes,
                qmll_workspace_bytes(grad ? QMLL_CALL_FORWARD_GRAD : QMLL_CALL_FORWARD, p, n_atoms, n_mol,
                                     (grad && grad->layout == QMLL_GRAD_DENSE) ? grad->dense_floats : 0));
  if (rc) return rc;
  Carver ws(workspace, workspace_bytes);
  SorfTables t;
  rc = sorf_prepare_tables(p, nullptr, ws, &t, st);
  if (rc) return rc;
  float* zs = grad ? ws.take<float>(sorf_zs_floats(p, n_atoms)) : nullptr;
  if (!ws.fits()) return QMLL_ERR_WORKSPACE;
  SorfProblem pr{p, x, elem, mol_off, n_atoms, n_mol};
  rc = sorf_launch_forward(pr, t, Z, zs, st);
  if (rc) return rc;
  if (grad) {
    if (grad->layout == QMLL_GRAD_DENSE && use_rows_mma(p, force_rows_mode)) {
      void* W16 = ws.take<uint8_t>(sorf_mma_w_bytes(p));
      const size_t xb = sorf_mma_x_bytes(p, n_atoms, grad->dense_floats);
      void* Xh = ws.take<uint8_t>(xb);
      void* Xl = ws.take<uint8_t>(xb);
      long long* xoff = ws.take<long long>((size_t)n_mol + 1);
      float* inv_scale = ws.take<float>((size_t)n_atoms);
      if (!ws.fits()) return QMLL_ERR_WORKSPACE;
      rc = sorf_force_rows_dense_mma(pr, t, zs, grad, W16, Xh, Xl, xoff, inv_scale, G, st,
                                     force_rows_mode != QMLL_ROWS_MMA);   // AUTO: CTA pairs
    } else if (grad->layout == QMLL_GRAD_DENSE) {
      float* gt = ws.take<float>((size_t)grad->dense_floats);
      if (!ws.fits()) return QMLL_ERR_WORKSPACE;
      rc = sorf_transpose_dense(pr, grad->dense, grad->dense_off, gt, st);
      if (rc) return rc;
      rc = sorf_launch_force_rows_dense(pr, t, zs, gt, grad->dense_off, G, st);
    } else {
      rc = sorf_launch_force_rows_neighbor(pr, t, zs, grad->nbr_idx, grad->nbr_val, grad->K, G, st);
    }
  }
  return rc;
}

int qmll_sorf_forward(const qmll_sorf_params* p, const float* x, const int32_t* elem, const int32_t* mol_off,
                      int64_t n_atoms, int32_t n_mol, const qmll_grad* grad, float* Z, float* G, void* workspace,
                      size_t workspace_bytes, void* cuda_stream) {
  return qmll_sorf_forward_mode(p, x, elem, mol_off, n_atoms, n_mol, grad, Z, G, workspace, workspace_bytes,
                                QMLL_ROWS_AUTO, cuda_stream);
}

size_t qmll_featmap_workspace_bytes(int32_t d, int32_t D, int32_t n_elem, int64_t n_atoms, int32_t rff) {
  if (d <= 0 || D <= 0 || n_elem <= 0 || n_atoms < 0) return 0;
  qmll_sorf_params q{d, D, 3, n_elem, 1.f, nullptr, nullptr};
  return featmap_mma_scratch_bytes(d, n_elem, n_atoms) + featmap_mma_w_bytes(d, D, n_elem, rff != 0) +
         (rff ? 0 : sorf_tables_bytes(&q, false)) + 1024;
}

int qmll_sorf_forward_mma(const qmll_sorf_params* p, const float* x, const int32_t* elem, const int32_t* mol_off,
                          int64_t n_atoms, int32_t n_mol, float* Z, void* workspace, size_t workspace_bytes,
                          void* cuda_stream) {
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int rc = check_params(p);
  if (rc) return rc;
  rc = check_problem(x, elem, mol_off, n_atoms, n_mol);
  if (rc) return rc;
  if (!Z) return QMLL_ERR_INVALID_ARG;
  if (!featmap_mma_supported(p->d, p->n_elem)) return QMLL_ERR_UNSUPPORTED;
  rc = check_device();
  if (rc) return rc;
  rc = check_ws(workspace, workspace_bytes, qmll_featmap_workspace_bytes(p->d, p->D, p->n_elem, n_atoms, 0));
  if (rc) return rc;
  Carver ws(workspace, workspace_bytes);
  SorfTables t;
  rc = sorf_prepare_tables(p, nullptr, ws, &t, st);
  if (rc) return rc;
  void* W16 = ws.take<uint8_t>(sorf_mma_w_bytes(p));
  if (!ws.fits()) return QMLL_ERR_WORKSPACE;
  rc = sorf_mma_build_w(p, t, W16, st);
  if (rc) return rc;
  SorfProblem pr{p, x, elem, mol_off, n_atoms, n_mol};
  return featmap_sorf_forward_mma(pr, W16, Z, ws, st);
}

int qmll_rff_forward(const float* W, const float* bias, int32_t d, int32_t D, int32_t n_elem, const float* x,
                     const int32_t* elem, const int32_t* mol_off, int64_t n_atoms, int32_t n_mol, float* Z,
                     void* workspace, size_t workspace_bytes, void* cuda_stream) {
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (!W || !bias || !Z || d <= 0 || D <= 0 || D % 4 != 0 || n_elem < 1) return QMLL_ERR_INVALID_ARG;
  int rc = check_problem(x, elem, mol_off, n_atoms, n_mol);
  if (rc) return rc;
  if (!featmap_mma_supported(d, n_elem)) return QMLL_ERR_UNSUPPORTED;
  rc = check_device();
  if (rc) return rc;
  rc = check_ws(workspace, workspace_bytes, qmll_featmap_workspace_bytes(d, D, n_elem, n_atoms, 1));
  if (rc) return rc;
  Carver ws(workspace, workspace_bytes);
  return featmap_rff_forward(W, bias, d, D, n_elem, x, elem, mol_off, n_atoms, n_mol, Z, ws, st);
}

int qmll_sorf_backward_forces(const qmll_sorf_params* p, const float* x, const int32_t* elem,
                              const int32_t* mol_off, int64_t n_atoms, int32_t n_mol, const float* alpha,
                              const qmll_grad* grad, float* forces, void* workspace, size_t workspace_bytes,
                              void* cuda_stream) {
  if (!forces || !grad) return QMLL_ERR_INVALID_ARG;
  return backward_impl(p, x, elem, mol_off, n_atoms, n_mol, alpha, grad, nullptr, forces, workspace,
                       workspace_bytes, static_cast<cudaStream_t>(cuda_stream), QMLL_CALL_BACKWARD_FORCES);
}

static int check_fchl(const qmll_fchl19_params* fp);

int qmll_sorf_backward_g(const qmll_sorf_params* p, const float* x, const int32_t* elem, const int32_t* mol_off,
                         int64_t n_atoms, int32_t n_mol, const float* alpha, float* energies, float* g,
                         void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!g) return QMLL_ERR_INVALID_ARG;
  return backward_impl(p, x, elem, mol_off, n_atoms, n_mol, alpha, nullptr, energies, nullptr, workspace,
                       workspace_bytes, static_cast<cudaStream_t>(cuda_stream), QMLL_CALL_PREDICT, g);
}

int qmll_project_back(const float* g, const int32_t* elem, int64_t n_atoms, int32_t rep, int32_t d, int32_t n_elem,
                      const float* U, float* w, void* cuda_stream) {
  if (n_atoms < 0 || rep <= 0 || d <= 0 || d % 4 != 0 || n_elem < 1 || !U) return QMLL_ERR_INVALID_ARG;
  if (n_atoms > 0 && (!g || !elem || !w)) return QMLL_ERR_INVALID_ARG;
  if (n_atoms > 0x7fffff00LL || d > 8192) return QMLL_ERR_INVALID_ARG;
  int rc = check_device();
  if (rc) return rc;
  return project_back_launch(g, elem, n_atoms, rep, d, n_elem, U, w, static_cast<cudaStream_t>(cuda_stream));
}

int qmll_fchl19_backward(const qmll_fchl19_params* fp, const float* r, const int32_t* elem, int64_t n_atoms,
                         const int32_t* nbr_idx, const float* nbr_shift, int32_t K, const float* w, float* forces,
                         int32_t* info, void* cuda_stream) {
  int rc = check_fchl(fp);
  if (rc) return rc;
  if (n_atoms < 0 || n_atoms > 0x7fffff00LL || K < 0 || K > 4096 || !info) return QMLL_ERR_INVALID_ARG;
  if (n_atoms > 0 && (!r || !elem || !w || !forces || (K > 0 && !nbr_idx))) return QMLL_ERR_INVALID_ARG;
  rc = check_device();
  if (rc) return rc;
  if (n_atoms == 0) return fchl19_launch(fp, r, elem, 0, nbr_idx, nbr_shift, K, nullptr, nullptr, nullptr, info, nullptr,
                                         nullptr, static_cast<cudaStream_t>(cuda_stream));
  return fchl19_launch(fp, r, elem, n_atoms, nbr_idx, nbr_shift, K, nullptr, nullptr, nullptr, info, w, forces,
                       static_cast<cudaStream_t>(cuda_stream));
}

int qmll_predict(const qmll_sorf_params* p, const float* x, const int32_t* elem, const int32_t* mol_off,
                 int64_t n_atoms, int32_t n_mol, const float* alpha, const qmll_grad* grad, float* energies,
                 float* forces, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!energies) return QMLL_ERR_INVALID_ARG;
  return backward_impl(p, x, elem, mol_off, n_atoms, n_mol, alpha, grad, energies, forces, workspace,
                       workspace_bytes, static_cast<cudaStream_t>(cuda_stream), QMLL_CALL_PREDICT);
}

int qmll_normal_equations_mode(const float* A, const float* y, int64_t rows, int32_t D, int32_t accumulate,
                               float* ZtZ, float* Zty, void* workspace, size_t workspace_bytes, int32_t mode,
                               void* cuda_stream) {
  if (rows < 0 || D <= 0 || !ZtZ || !valid_mode(mode)) return QMLL_ERR_INVALID_ARG;
  if (rows > 0 && !A) return QMLL_ERR_INVALID_ARG;
  if (rows > 0 && (y != nullptr) != (Zty != nullptr)) return QMLL_ERR_INVALID_ARG;
  int rc = check_device();
  if (rc) return rc;
  return syrk_normal_equations(A, y, rows, D, accumulate, ZtZ, Zty, workspace, workspace_bytes, mode,
                               static_cast<cudaStream_t>(cuda_stream));
}

int qmll_normal_equations(const float* A, const float* y, int64_t rows, int32_t D, int32_t accumulate, float* ZtZ,
                          float* Zty, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  return qmll_normal_equations_mode(A, y, rows, D, accumulate, ZtZ, Zty, workspace, workspace_bytes,
                                    QMLL_NE_SPLIT_F16, cuda_stream);
}

int qmll_project(const float* rho, const int32_t* elem, const int32_t* mol_off, int64_t n_atoms, int32_t n_mol,
                 int32_t rep, int32_t d, int32_t n_elem, const float* U, float* x, const float* grad_in,
                 const int64_t* grad_in_off, float* grad_out, const int64_t* grad_out_off, void* cuda_stream) {
  if (n_atoms < 0 || n_mol < 0 || rep <= 0 || d <= 0 || d % 4 != 0 || n_elem < 1 || !U) return QMLL_ERR_INVALID_ARG;
  if (!x && !grad_out) return QMLL_ERR_INVALID_ARG;
  if (n_atoms > 0 && (!elem || (x && !rho))) return QMLL_ERR_INVALID_ARG;
  if (grad_out && (!grad_in || !grad_in_off || !grad_out_off || !mol_off || n_atoms > 0x7fffff00LL))
    return QMLL_ERR_INVALID_ARG;
  int rc = check_device();
  if (rc) return rc;
  return project_launch(rho, elem, mol_off, n_atoms, n_mol, rep, d, n_elem, U, x, grad_in, grad_in_off, grad_out,
                        grad_out_off, static_cast<cudaStream_t>(cuda_stream));
}

int qmll_project_neighbor(const float* grad_in, const int32_t* idx, const int32_t* elem, int64_t n_atoms, int32_t S,
                          int32_t rep, int32_t d, int32_t n_elem, const float* U, float* grad_out,
                          void* cuda_stream) {
  if (n_atoms < 0 || S < 0 || rep <= 0 || d <= 0 || d % 4 != 0 || n_elem < 1 || !U) return QMLL_ERR_INVALID_ARG;
  if (n_atoms > 0 && S > 0 && (!grad_in || !grad_out || !elem)) return QMLL_ERR_INVALID_ARG;
  if (n_atoms * (int64_t)S > 0x7fffff00LL) return QMLL_ERR_INVALID_ARG;
  int rc = check_device();
  if (rc) return rc;
  return project_neighbor_launch(grad_in, idx, elem, n_atoms, S, rep, d, n_elem, U, grad_out,
                                 static_cast<cudaStream_t>(cuda_stream));
}

static int check_fchl(const qmll_fchl19_params* fp) {
  if (!fp) return QMLL_ERR_INVALID_ARG;
  if (fp->n_elem < 1 || fp->n2 < 1 || fp->n3 < 1) return QMLL_ERR_INVALID_ARG;
  if (!(fp->eta2 > 0.f) || !(fp->eta3 > 0.f) || !(fp->r_cut > 0.f)) return QMLL_ERR_INVALID_ARG;
  if (fp->n_elem > 16 || fp->n2 > 32 || fp->n3 > 32) return QMLL_ERR_UNSUPPORTED;
  return QMLL_OK;
}

int32_t qmll_fchl19_rep_size(const qmll_fchl19_params* fp) { return check_fchl(fp) ? -1 : fchl19_rep_size(fp); }

int qmll_fchl19(const qmll_fchl19_params* fp, const float* r, const int32_t* elem, int64_t n_atoms,
                const int32_t* nbr_idx, const float* nbr_shift, int32_t K, float* rho, int32_t* jac_idx,
                float* jac_val, int32_t* info, void* cuda_stream) {
  int rc = check_fchl(fp);
  if (rc) return rc;
  if (n_atoms < 0 || n_atoms > 0x7fffff00LL || K < 0 || K > 4096 || !info) return QMLL_ERR_INVALID_ARG;
  if (n_atoms > 0 && ((jac_idx == nullptr) != (jac_val == nullptr) || (!rho && !jac_val))) return QMLL_ERR_INVALID_ARG;
  if (n_atoms > 0 && (!r || !elem || (K > 0 && !nbr_idx))) return QMLL_ERR_INVALID_ARG;
  rc = check_device();
  if (rc) return rc;
  return fchl19_launch(fp, r, elem, n_atoms, nbr_idx, nbr_shift, K, rho, jac_idx, jac_val, info, nullptr, nullptr,
                       static_cast<cudaStream_t>(cuda_stream));
}

int qmll_pack_lower(const float* ZtZ, int32_t D, float* packed, void* cuda_stream) {
  if (!ZtZ || !packed || D <= 0 || D > 65535) return QMLL_ERR_INVALID_ARG;
  int rc = check_device();
  if (rc) return rc;
  return syrk_pack_lower(ZtZ, D, packed, static_cast<cudaStream_t>(cuda_stream));
}
int qmll_unpack_lower(const float* packed, int32_t D, float* ZtZ, void* cuda_stream) {
  if (!ZtZ || !packed || D <= 0 || D > 65535) return QMLL_ERR_INVALID_ARG;
  int rc = check_device();
  if (rc) return rc;
  return syrk_unpack_lower(packed, D, ZtZ, static_cast<cudaStream_t>(cuda_stream));
}

int qmll_energies(const float* Z, const float* alpha, int64_t n_mol, int32_t D, float* energies, void* cuda_stream) {
  if (n_mol < 0 || D <= 0 || !alpha || (n_mol > 0 && (!Z || !energies))) return QMLL_ERR_INVALID_ARG;
  int rc = check_device();
  if (rc) return rc;
  return energies_from_z(Z, alpha, n_mol, D, energies, static_cast<cudaStream_t>(cuda_stream));
}

int qmll_solve(const float* ZtZ, const float* Zty, int32_t D, double lambda, float* alpha, int32_t* info,
               void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!ZtZ || !Zty || !alpha || !info || D <= 0 || !(lambda >= 0.0)) return QMLL_ERR_INVALID_ARG;
  int rc = check_device();
  if (rc) return rc;
  return solve_normal_equations(ZtZ, Zty, D, lambda, alpha, info, workspace, workspace_bytes,
                                static_cast<cudaStream_t>(cuda_stream));
}

const char* qmll_status_string(int status) {
  static thread_local char buf[640];
  switch (status) {
    case QMLL_OK: return "QMLL_OK";
    case QMLL_ERR_INVALID_ARG: return "QMLL_ERR_INVALID_ARG: invalid argument";
    case QMLL_ERR_UNSUPPORTED: return "QMLL_ERR_UNSUPPORTED: unsupported size or device (needs sm_100, d in 16..1024)";
    case QMLL_ERR_WORKSPACE: return "QMLL_ERR_WORKSPACE: workspace missing, misaligned or too small";
    case QMLL_ERR_CUDA:
      snprintf(buf, sizeof(buf), "QMLL_ERR_CUDA: %s", g_err_text);
      return buf;
    default: return "unknown qmll status";
  }
}

void qmll_time_normal_equations_kernel(int enable) { syrk_set_timing(enable != 0); }
int qmll_collect_normal_equations_kernel_ms(double* total_ms, int* launches) {
  if (!total_ms || !launches) return QMLL_ERR_INVALID_ARG;
  return syrk_collect_timing(total_ms, launches);
}

int64_t qmll_launch_count(void) { return g_launches.load(); }
void qmll_reset_launch_count(void) { g_launches.store(0); }

}  // extern "C"
