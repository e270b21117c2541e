// energy_kernels.cu -- qmll_energies: E[M] = sum_l Z[M, l] alpha[l]  (eq. 15: the prediction is linear
// in the summed features), for callers that already hold Z -- the training matrix, or the output of the tensor-core
// feature map (qmll_sorf_forward_mma / qmll_rff_forward), which makes "feature map on tcgen05 + this pass" the
// energies-only prediction of the f4 variants.  One streaming pass over Z: HBM-bound, 4 D bytes per molecule.
// Warp = molecule row: 16-byte loads, four fp32 partial sums per lane (D / 128 terms each), combined in FP64.
#include "qmll_common.cuh"

namespace qmll {

int device_sm_count();   // sorf_dispatch.cu

__global__ void __launch_bounds__(256)
energies_from_z_kernel(const float* __restrict__ Z, const float* __restrict__ alpha, long long n_mol, int D,
                       float* __restrict__ energies) {
  const int lane = threadIdx.x & 31;
  const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const long long n_warps = ((long long)gridDim.x * blockDim.x) >> 5;
  const bool vec = (D & 3) == 0 && ((uintptr_t)Z & 15) == 0 && ((uintptr_t)alpha & 15) == 0;
  for (long long M = warp0; M < n_mol; M += n_warps) {
    const float* row = Z + (size_t)M * D;
    float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
    if (vec) {
      const float4* r4 = reinterpret_cast<const float4*>(row);
      const float4* a4 = reinterpret_cast<const float4*>(alpha);
#pragma unroll 4
      for (int q = lane; q < D / 4; q += 32) {
        const float4 z = __ldcs(r4 + q);
        const float4 a = __ldg(a4 + q);
        s0 = fmaf(z.x, a.x, s0); s1 = fmaf(z.y, a.y, s1); s2 = fmaf(z.z, a.z, s2); s3 = fmaf(z.w, a.w, s3);
      }
    } else {
      for (int l = lane; l < D; l += 32) s0 = fmaf(__ldcs(row + l), __ldg(alpha + l), s0);
    }
    double s = ((double)s0 + (double)s1) + ((double)s2 + (double)s3);
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) s += __shfl_xor_sync(0xffffffffu, s, m);
    if (lane == 0) energies[M] = (float)s;
  }
}

int energies_from_z(const float* Z, const float* alpha, int64_t n_mol, int32_t D, float* energies, cudaStream_t st) {
  if (n_mol == 0) return QMLL_OK;
  const long long want = (n_mol + 7) / 8;                      // 8 warps per block, one row per warp and pass
  const long long cap = (long long)device_sm_count() * 16;
  const unsigned blocks = (unsigned)(want < cap ? want : cap);
  energies_from_z_kernel<<<blocks, 256, 0, st>>>(Z, alpha, n_mol, D, energies);
  QMLL_LAUNCH_CHECK("energies_from_z_kernel");
  return QMLL_OK;
}

}  // namespace qmll
