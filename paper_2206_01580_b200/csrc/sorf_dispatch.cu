// sorf_dispatch.cu -- table packing kernels, workspace layout of the packed tables and the switch over the
// supported descriptor lengths (the kernels themselves are instantiated in sorf_d*.cu).
#include "sorf_kernels.cuh"

namespace qmll {

// ------------------------------------------------------------------------------------------------
// Table packing: the per-(element, stack group) lane-ordered layouts documented in sorf_device.cuh.
// ------------------------------------------------------------------------------------------------
__global__ void pack_signs_kernel(const int8_t* __restrict__ signs, uint32_t* __restrict__ out, int n_elem,
                                  int n_s, int n_sg, int T, int d, int E, int P, int EW) {
  const int spw = kWarp / P;
  const long long total = (long long)n_elem * T * n_sg * EW * kWarp;
  for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
       idx += (long long)gridDim.x * blockDim.x) {
    const int lane = (int)(idx % kWarp);
    long long r = idx / kWarp;
    const int k = (int)(r % EW); r /= EW;
    const int sg = (int)(r % n_sg); r /= n_sg;
    const int t = (int)(r % T);
    const int e = (int)(r / T);
    const int s = sg * spw + lane / P, p = lane % P;
    uint32_t w = 0;
    if (s < n_s) {
      const int8_t* src = signs + (((size_t)e * n_s + s) * T + t) * d + p * E + 32 * k;
      const int nb = E - 32 * k < 32 ? E - 32 * k : 32;
      for (int i = 0; i < nb; ++i) w |= (src[i] < 0 ? 1u : 0u) << i;
    }
    out[idx] = w;
  }
}

__global__ void permute_table_kernel(const float* __restrict__ in /* [rows, D] */, float* __restrict__ out,
                                     int rows, int n_s, int n_sg, int d, int E, int P, float scale) {
  const int E4 = E / 4, spw = kWarp / P;
  const long long D = (long long)n_s * d;
  const long long total = (long long)rows * n_sg * E4 * kWarp * 4;
  for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
       idx += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(idx & 3);
    long long r = idx >> 2;
    const int lane = (int)(r % kWarp); r /= kWarp;
    const int q = (int)(r % E4); r /= E4;
    const int sg = (int)(r % n_sg);
    const int e = (int)(r / n_sg);
    const int s = sg * spw + lane / P, p = lane % P;
    out[idx] = s < n_s ? in[e * D + (long long)s * d + p * E + 4 * q + i] * scale : 0.f;
  }
}


__global__ void finish_energies_kernel(const double* __restrict__ acc, float* __restrict__ out, int n) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = (float)acc[i];
}

// Dense gradient [n, d, n, 3] = (I, m, j, k)  ->  [n, n, 3, d] = (I, j, k, m) per molecule: every gradient column
// becomes d contiguous floats (what the force-row kernel stages with one bulk copy).  Block = one atom I: a
// [d, 3n] -> [3n, d] transposition through 32 x 96 shared-memory tiles, coalesced on both sides.
__global__ void __launch_bounds__(256)
transpose_dense_kernel(const float* __restrict__ dense, const int64_t* __restrict__ dense_off,
                       const int32_t* __restrict__ mol_off, int n_mol, int d, float* __restrict__ gt) {
  __shared__ float tile[32][97];
  const int Ig = blockIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int M = owner_molecule(mol_off, n_mol, Ig);
  const int a0 = __ldg(mol_off + M), n = __ldg(mol_off + M + 1) - a0;
  const int ncol = 3 * n;
  const size_t base = (size_t)__ldg(dense_off + M) + (size_t)(Ig - a0) * d * ncol;
  const float* src = dense + base;  // [d][ncol]
  float* dst = gt + base;           // [ncol][d]
  for (int c0 = 0; c0 < ncol; c0 += 96) {
    const int nc = ncol - c0 < 96 ? ncol - c0 : 96;
    for (int m0 = 0; m0 < d; m0 += 32) {
      const int nm = d - m0 < 32 ? d - m0 : 32;
      __syncthreads();
      for (int rr = warp; rr < nm; rr += 8)
        for (int cc = lane; cc < nc; cc += 32) tile[rr][cc] = __ldcs(src + (size_t)(m0 + rr) * ncol + c0 + cc);
      __syncthreads();
      for (int cc = warp; cc < nc; cc += 8)
        if (lane < nm) dst[(size_t)(c0 + cc) * d + m0 + lane] = tile[lane][cc];
    }
  }
}

int sorf_transpose_dense(const SorfProblem& pr, const float* dense, const int64_t* dense_off, float* gt,
                         cudaStream_t st) {
  if (pr.n_atoms == 0) return QMLL_OK;
  transpose_dense_kernel<<<(unsigned)pr.n_atoms, 256, 0, st>>>(dense, dense_off, pr.mol_off, pr.n_mol, pr.p->d, gt);
  QMLL_LAUNCH_CHECK("transpose_dense_kernel");
  return QMLL_OK;
}

int device_sm_count() {
  static int cached = 0;
  if (cached == 0) {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0)
      cached = n;
    else
      return 148;
  }
  return cached;
}

bool sorf_supported_d(int d) { return d >= 16 && d <= 1024 && (d & (d - 1)) == 0; }

static void shape_of(int d, int* E, int* P) {
  *E = shape_E(d);
  *P = shape_P(d);
}

// floats of the per-atom sin table written by the forward kernel: [n_atoms][n_sg][E*32]
size_t sorf_zs_floats(const qmll_sorf_params* p, int64_t n_atoms) {
  int E, P;
  shape_of(p->d, &E, &P);
  const int spw = kWarp / P, n_s = p->D / p->d, n_sg = (n_s + spw - 1) / spw;
  return (size_t)n_atoms * n_sg * E * kWarp;
}

size_t sorf_tables_bytes(const qmll_sorf_params* p, bool with_alpha) {
  int E, P;
  shape_of(p->d, &E, &P);
  const size_t spw = kWarp / P, n_s = p->D / p->d, n_sg = (n_s + spw - 1) / spw, EW = (E + 31) / 32;
  size_t b = align_up((size_t)p->n_elem * p->n_transform * n_sg * EW * kWarp * 4, 256);
  b += align_up((size_t)p->n_elem * n_sg * E * kWarp * 4, 256);
  if (with_alpha) b += align_up(n_sg * E * kWarp * 4, 256);
  return b + 256;
}

int sorf_prepare_tables(const qmll_sorf_params* p, const float* alpha, Carver& ws, SorfTables* t,
                        cudaStream_t st) {
  int E, P;
  shape_of(p->d, &E, &P);
  const int spw = kWarp / P, n_s = p->D / p->d, n_sg = (n_s + spw - 1) / spw, EW = (E + 31) / 32;
  const size_t n_sign = (size_t)p->n_elem * p->n_transform * n_sg * EW * kWarp;
  const size_t n_tab = (size_t)n_sg * E * kWarp;
  t->sign_bits = ws.take<uint32_t>(n_sign);
  t->bias_t = ws.take<float>((size_t)p->n_elem * n_tab);
  t->alpha_s = alpha ? ws.take<float>(n_tab) : nullptr;
  if (!ws.fits()) return QMLL_ERR_WORKSPACE;
  const int threads = 256;
  auto blocks = [&](size_t n) { size_t b = (n + threads - 1) / threads; return (unsigned)(b > 65535 ? 65535 : (b ? b : 1)); };
  pack_signs_kernel<<<blocks(n_sign), threads, 0, st>>>(p->signs, t->sign_bits, p->n_elem, n_s, n_sg, p->n_transform,
                                                        p->d, E, P, EW);
  QMLL_LAUNCH_CHECK("pack_signs_kernel");
  permute_table_kernel<<<blocks((size_t)p->n_elem * n_tab), threads, 0, st>>>(p->bias, t->bias_t, p->n_elem, n_s, n_sg,
                                                                              p->d, E, P, 1.0f);
  QMLL_LAUNCH_CHECK("permute_table_kernel(bias)");
  if (alpha) {
    permute_table_kernel<<<blocks(n_tab), threads, 0, st>>>(alpha, t->alpha_s, 1, n_s, n_sg, p->d, E, P,
                                                            (float)sqrt(2.0 / (double)p->D));
    QMLL_LAUNCH_CHECK("permute_table_kernel(alpha)");
  }
  return QMLL_OK;
}

#define QMLL_SWITCH_D(d, CALL)                    \
  switch (d) {                                    \
    case 16: return CALL(d16);                    \
    case 32: return CALL(d32);                    \
    case 64: return CALL(d64);                    \
    case 128: return CALL(d128);                  \
    case 256: return CALL(d256);                  \
    case 512: return CALL(d512);                  \
    case 1024: return CALL(d1024);                \
    default: return QMLL_ERR_UNSUPPORTED;         \
  }

int sorf_launch_forward(const SorfProblem& pr, const SorfTables& t, float* Z, float* zs_out, cudaStream_t st) {
#define CALL(TAG) sorf_forward_##TAG(pr, t, Z, zs_out, st)
  QMLL_SWITCH_D(pr.p->d, CALL)
#undef CALL
}
// forces: [n_atoms, 3] with grad, or (grad == NULL, g_out = true) g [n_atoms, d] = dE/dx
int sorf_launch_predict(const SorfProblem& pr, const SorfTables& t, const qmll_grad* grad, float* forces,
                        double* energy_acc, cudaStream_t st, bool g_out) {
  GradView gv{QMLL_GRAD_NONE, nullptr, nullptr, nullptr, nullptr, 0};
  if (grad) gv = GradView{grad->layout, grad->dense, grad->dense_off, grad->nbr_idx, grad->nbr_val, grad->K};
  if (g_out) gv.layout = kGradGOut;
#define CALL(TAG) sorf_predict_##TAG(pr, t, gv, forces, energy_acc, st)
  QMLL_SWITCH_D(pr.p->d, CALL)
#undef CALL
}
int sorf_launch_force_rows_dense(const SorfProblem& pr, const SorfTables& t, const float* zs,
                                 const float* dense_t, const int64_t* dense_off, float* G, cudaStream_t st) {
#define CALL(TAG) sorf_force_rows_dense_##TAG(pr, t, zs, dense_t, dense_off, G, st)
  QMLL_SWITCH_D(pr.p->d, CALL)
#undef CALL
}
int sorf_launch_force_rows_neighbor(const SorfProblem& pr, const SorfTables& t, const float* zs,
                                    const int32_t* nbr_idx, const float* nbr_val, int K, float* G,
                                    cudaStream_t st) {
#define CALL(TAG) sorf_force_rows_neighbor_##TAG(pr, t, zs, nbr_idx, nbr_val, K, G, st)
  QMLL_SWITCH_D(pr.p->d, CALL)
#undef CALL
}

int sorf_finish_energies(const double* energy_acc, float* energies, int32_t n_mol, cudaStream_t st) {
  if (n_mol == 0) return QMLL_OK;
  finish_energies_kernel<<<(n_mol + 255) / 256, 256, 0, st>>>(energy_acc, energies, n_mol);
  QMLL_LAUNCH_CHECK("finish_energies_kernel");
  return QMLL_OK;
}

}  // namespace qmll
