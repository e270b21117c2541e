// qmll_common.cuh -- shared host-side plumbing of the CUDA library (error handling, launch counter,
// workspace carving).  Internal to paper_2206_01580_b200/csrc; never included by oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/qmll.h"
#include "../../include/qmll_aux.h"

namespace qmll {

// Records the last CUDA error text for qmll_status_string (thread-local).
void note_cuda_error(cudaError_t err, const char* where);
void count_launch(int n = 1);

#define QMLL_CUDA_TRY(expr)                                  \
  do {                                                       \
    cudaError_t _e = (expr);                                 \
    if (_e != cudaSuccess) {                                 \
      ::qmll::note_cuda_error(_e, #expr);                    \
      return QMLL_ERR_CUDA;                                  \
    }                                                        \
  } while (0)

// After a kernel launch: counts it and turns a launch error into QMLL_ERR_CUDA.
#define QMLL_LAUNCH_CHECK(name)                              \
  do {                                                       \
    ::qmll::count_launch();                                  \
    cudaError_t _e = cudaGetLastError();                     \
    if (_e != cudaSuccess) {                                 \
      ::qmll::note_cuda_error(_e, name);                     \
      return QMLL_ERR_CUDA;                                  \
    }                                                        \
  } while (0)

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Bump allocator over the caller's workspace; `fits()` tells whether everything carved so far fits.
struct Carver {
  char* base;
  size_t size;
  size_t used = 0;
  Carver(void* b, size_t s) : base(static_cast<char*>(b)), size(s) {}
  template <typename T>
  T* take(size_t count) {
    size_t off = align_up(used, 256);
    used = off + count * sizeof(T);
    return reinterpret_cast<T*>(base ? base + off : nullptr);
  }
  bool fits() const { return used <= size; }
};

// ---- SORF (sorf_kernels.cu) ----------------------------------------------------------------------
struct SorfProblem {
  const qmll_sorf_params* p;
  const float* x;
  const int32_t* elem;
  const int32_t* mol_off;
  int64_t n_atoms;
  int32_t n_mol;
};

// Lane-ordered copies of the model tables living in the workspace (layouts in sorf_device.cuh).
struct SorfTables {
  uint32_t* sign_bits;  // [n_elem][T][n_sg][EW][32]
  float* bias_t;        // [n_elem][n_sg][E/4][32][4]   bias (radians)
  float* alpha_s;       // [n_sg][E/4][32][4]           alpha * sqrt(2/D)   (may be unused)
};

size_t sorf_tables_bytes(const qmll_sorf_params* p, bool with_alpha);
int sorf_prepare_tables(const qmll_sorf_params* p, const float* alpha, Carver& ws, SorfTables* t,
                        cudaStream_t st);
int sorf_launch_forward(const SorfProblem& pr, const SorfTables& t, float* Z, float* zs_out, cudaStream_t st);
int sorf_launch_predict(const SorfProblem& pr, const SorfTables& t, const qmll_grad* grad, float* forces,
                        double* energy_acc, cudaStream_t st, bool g_out = false);
int sorf_launch_force_rows_dense(const SorfProblem& pr, const SorfTables& t, const float* zs,
                                 const float* dense_t, const int64_t* dense_off, float* G, cudaStream_t st);
size_t sorf_zs_floats(const qmll_sorf_params* p, int64_t n_atoms);

// ---- force rows on the tensor cores (sorf_mma.cu) -----------------------------------------------------
bool sorf_mma_supported(const qmll_sorf_params* p);
size_t sorf_mma_w_bytes(const qmll_sorf_params* p);
size_t sorf_mma_x_bytes(const qmll_sorf_params* p, int64_t n_atoms, int64_t dense_floats);
int sorf_force_rows_dense_mma(const SorfProblem& pr, const SorfTables& t, const float* zs, const qmll_grad* grad,
                              void* W16, void* Xh, void* Xl, long long* xoff, float* inv_scale, float* G,
                              cudaStream_t st, bool pairs = false);
int sorf_mma_build_w(const qmll_sorf_params* p, const SorfTables& t, void* W16, cudaStream_t st);

// ---- feature map on the tensor cores (featmap_mma.cu): SORF with expanded W, dense-W RFF ----------------------------
bool featmap_mma_supported(int d, int n_elem);
size_t featmap_mma_scratch_bytes(int d, int n_elem, int64_t n_atoms);
size_t featmap_mma_w_bytes(int d, int D, int n_elem, bool rff);
int featmap_sorf_forward_mma(const SorfProblem& pr, const void* W16, float* Z, Carver& ws, cudaStream_t st);
int featmap_rff_forward(const float* W, const float* bias, int d, int D, int n_elem, const float* x, const int32_t* elem,
                        const int32_t* mol_off, int64_t n_atoms, int32_t n_mol, float* Z, Carver& ws, cudaStream_t st);

int sorf_launch_force_rows_neighbor(const SorfProblem& pr, const SorfTables& t, const float* zs,
                                    const int32_t* nbr_idx, const float* nbr_val, int K, float* G,
                                    cudaStream_t st);
int sorf_transpose_dense(const SorfProblem& pr, const float* dense, const int64_t* dense_off, float* gt,
                         cudaStream_t st);
int sorf_finish_energies(const double* energy_acc, float* energies, int32_t n_mol, cudaStream_t st);
bool sorf_supported_d(int d);

// ---- normal equations (syrk_tcgen05.cu) ----------------------------------------------------------------
size_t syrk_min_workspace(int32_t D, int mode);
size_t syrk_full_workspace(int64_t rows, int32_t D, int mode);
int syrk_normal_equations(const float* A, const float* y, int64_t rows, int32_t D, int accumulate, float* ZtZ,
                          float* Zty, void* ws, size_t ws_bytes, int mode, cudaStream_t st);

int syrk_pack_lower(const float* C, int32_t D, float* packed, cudaStream_t st);
int syrk_unpack_lower(const float* packed, int32_t D, float* C, cudaStream_t st);

// ---- solve (solve_kernels.cu) ------------------------------------------------------------------------------
int energies_from_z(const float* Z, const float* alpha, int64_t n_mol, int32_t D, float* energies, cudaStream_t st);
size_t solve_workspace_bytes(int32_t D);
int solve_normal_equations(const float* ZtZ, const float* Zty, int32_t D, double lambda, float* alpha, int32_t* info,
                           void* ws, size_t ws_bytes, cudaStream_t st);

// ---- per-element PCA projection (project_kernels.cu) ------------------------------------------------------
int project_launch(const float* rho, const int32_t* elem, const int32_t* mol_off, int64_t n_atoms, int32_t n_mol,
                   int32_t rep, int32_t d, int32_t n_elem, const float* U, float* x, const float* gin,
                   const int64_t* in_off, float* gout, const int64_t* out_off, cudaStream_t st);

int project_back_launch(const float* g, const int32_t* elem, int64_t n_atoms, int32_t rep, int32_t d, int32_t n_elem,
                        const float* U, float* w, cudaStream_t st);
int project_neighbor_launch(const float* gin, const int32_t* idx, const int32_t* elem, int64_t n_atoms, int32_t S,
                            int32_t rep, int32_t d, int32_t n_elem, const float* U, float* gout, cudaStream_t st);

// ---- FCHL19 representation and Jacobian (fchl19_kernels.cu) --------------------------------------------------
int fchl19_rep_size(const qmll_fchl19_params* fp);
int fchl19_launch(const qmll_fchl19_params* fp, const float* r, const int32_t* elem, int64_t n_atoms,
                  const int32_t* nbr_idx, const float* nbr_shift, int32_t K, float* rho, int32_t* jac_idx,
                  float* jac_val, int32_t* info, const float* w_in, float* forces, cudaStream_t st);

void syrk_set_timing(bool on);
int syrk_collect_timing(double* total_ms, int* launches);

}  // namespace qmll
