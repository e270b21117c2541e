// predict_static.cu -- qmll_predict_static: qmll_predict (energies E = Z alpha,
// PAPER.md eq. 14-15, and forces, L137 / eq. 17) for callers that cannot allocate device memory -- code
// under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The scratch qmll_predict takes as
// its `workspace` argument (the lane-permuted sign / bias / alpha tables of the model and the FP64 energy
// accumulators, qmll_workspace_bytes(QMLL_CALL_PREDICT, ...)) lives here in a file-scope device array of
// QMLL_PREDICT_STATIC_MAX_BYTES; every GPU that loads the library holds it until the process exits.
//
// The array's name is a host-side stand-in in host code, NOT a device address: its device address is taken once per
// device with cudaGetSymbolAddress (that device current) and handed to the same kernels qmll_predict launches.
// Nothing here calls cudaMalloc / cudaFree or an allocating library routine; what must start at zero (the energy
// accumulators, the forces) is cleared by cudaMemsetAsync on the caller's stream in every call, and the tables are
// rewritten in full, so the contents a previous call left behind are never read.  All calls on a device SHARE the
// array: two calls that overlap on the GPU (different streams, no ordering between them) race.
#include <mutex>

#include "qmll_common.cuh"

namespace qmll {

static __device__ __align__(256) unsigned char g_predict_static_scratch[QMLL_PREDICT_STATIC_MAX_BYTES];

constexpr int kStaticMaxDevices = 64;
static std::mutex g_static_mutex;
static void* g_static_ptr[kStaticMaxDevices];   // device address of the array on every device, nullptr = not set up

// Once per device, with that device current: the device address of g_predict_static_scratch.
static int predict_static_scratch(void** out) {
  int dev = 0;
  QMLL_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kStaticMaxDevices) return QMLL_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (g_static_ptr[dev] == nullptr) {
    void* ptr = nullptr;
    QMLL_CUDA_TRY(cudaGetSymbolAddress(&ptr, g_predict_static_scratch));
    if (ptr == nullptr || ((uintptr_t)ptr & 255) != 0) return QMLL_ERR_CUDA;
    g_static_ptr[dev] = ptr;
  }
  *out = g_static_ptr[dev];
  return QMLL_OK;
}

}  // namespace qmll

using namespace qmll;

extern "C" {

size_t qmll_predict_static_max_bytes(void) { return (size_t)QMLL_PREDICT_STATIC_MAX_BYTES; }

int qmll_predict_static(const qmll_sorf_params* p, const float* x, const int32_t* elem, const int32_t* mol_off,
                        int64_t n_atoms, int32_t n_mol, const float* alpha, const qmll_grad* grad, float* energies,
                        float* forces, void* cuda_stream) {
  if (!p) return QMLL_ERR_INVALID_ARG;
  const size_t need = qmll_workspace_bytes(QMLL_CALL_PREDICT, p, n_atoms, n_mol, 0);
  if (need == 0) return QMLL_ERR_INVALID_ARG;                              // parameters qmll_predict rejects as well
  if (need > (size_t)QMLL_PREDICT_STATIC_MAX_BYTES) return QMLL_ERR_WORKSPACE;   // model / batch beyond the static scratch
  void* scratch = nullptr;
  const int rc = predict_static_scratch(&scratch);
  if (rc) return rc;
  return qmll_predict(p, x, elem, mol_off, n_atoms, n_mol, alpha, grad, energies, forces, scratch,
                      (size_t)QMLL_PREDICT_STATIC_MAX_BYTES, cuda_stream);
}

}  // extern "C"
