// contract_kernels.cu -- step a6: F[j,k] = -sum_I sum_m g_I[m] * d x_I[m] / d r_{j,k}  (F = -dE/dr, PAPER.md
// eq. 5/10 L63, L90), streaming the descriptor gradient exactly once.  HBM-bound: 2 flop per 4 B.
//   dense    (A12): per molecule a [n*d, 3n] matrix; F_M = -(g_M^T dx_M), a skinny GEMV.
//   neighbor (A13): per (I, q) a [d, 3] block scattered to atom j = nbr_idx[I, q] (duplicates accumulate).
#include "qmll_common.cuh"

namespace qmll {

constexpr int kCtrThreads = 256;

// Block (M, split): rows [r0, r1) of molecule M's [n*d, 3n] matrix.  Thread t owns column t % 3n and every
// RL-th row, so consecutive threads read consecutive floats of a row (rows are back to back in memory).
__global__ void __launch_bounds__(kCtrThreads)
contract_dense_kernel(const float* __restrict__ g, const int32_t* __restrict__ mol_off, int d,
                      const float* __restrict__ dense, const int64_t* __restrict__ dense_off,
                      float* __restrict__ forces, int splits) {
  __shared__ float sacc[kCtrThreads];
  const int M = blockIdx.x, split = blockIdx.y, t = threadIdx.x;
  const int a0 = __ldg(mol_off + M), n = __ldg(mol_off + M + 1) - a0;
  if (n <= 0) return;
  const int ncol = 3 * n;
  const long long nrow = (long long)n * d;
  const long long per = (nrow + splits - 1) / splits;
  const long long r0 = split * per, r1 = (r0 + per < nrow) ? r0 + per : nrow;
  if (r0 >= r1) return;
  const float* dx = dense + __ldg(dense_off + M);
  const float* gM = g + (size_t)a0 * d;

  if (ncol <= kCtrThreads) {
    const int RL = kCtrThreads / ncol;
    const int col = t % ncol, rl = t / ncol;
    sacc[t] = 0.f;
    __syncthreads();
    float acc = 0.f;
    if (rl < RL) {
      const float* ptr = dx + (size_t)col;
      long long r = r0 + rl;
      float acc2 = 0.f;
      // 8 independent streaming loads in flight per thread (the loop is HBM-latency bound otherwise)
      for (; r + 7LL * RL < r1; r += 8LL * RL) {
        float a[8], gv[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) a[u] = __ldcs(ptr + (size_t)(r + (long long)u * RL) * ncol);
#pragma unroll
        for (int u = 0; u < 8; ++u) gv[u] = __ldg(gM + r + (long long)u * RL);
#pragma unroll
        for (int u = 0; u < 8; u += 2) {
          acc = fmaf(gv[u], a[u], acc);
          acc2 = fmaf(gv[u + 1], a[u + 1], acc2);
        }
      }
      for (; r < r1; r += RL) acc = fmaf(__ldg(gM + r), __ldcs(ptr + (size_t)r * ncol), acc);
      atomicAdd(&sacc[col], acc + acc2);
    }
    __syncthreads();
    if (t < ncol) atomicAdd(forces + (size_t)a0 * 3 + t, -sacc[t]);
  } else {
    for (int col = t; col < ncol; col += kCtrThreads) {
      float acc = 0.f;
#pragma unroll 8
      for (long long r = r0; r < r1; ++r) acc = fmaf(__ldg(gM + r), __ldg(dx + (size_t)r * ncol + col), acc);
      atomicAdd(forces + (size_t)a0 * 3 + col, -acc);
    }
  }
}

// One warp per (I, q) pair: the [d, 3] block is 3d contiguous floats; a lane takes 12 of them (4 values of
// m times x, y, z) per step as three float4 loads.
__global__ void __launch_bounds__(kCtrThreads)
contract_neighbor_kernel(const float* __restrict__ g, long long n_pairs, int d, int K,
                         const int32_t* __restrict__ nbr_idx, const float* __restrict__ nbr_val,
                         float* __restrict__ forces) {
  const int lane = threadIdx.x & 31;
  const long long warp0 = ((long long)blockIdx.x * kCtrThreads + threadIdx.x) >> 5;
  const long long n_warps = ((long long)gridDim.x * kCtrThreads) >> 5;
  const int groups = d >> 2;
  for (long long pair = warp0; pair < n_pairs; pair += n_warps) {
    const int j = __ldg(nbr_idx + pair);
    if (j < 0) continue;
    const long long I = pair / K;
    const float4* val = reinterpret_cast<const float4*>(nbr_val + (size_t)pair * d * 3);
    const float4* g4 = reinterpret_cast<const float4*>(g + (size_t)I * d);
    float ax = 0.f, ay = 0.f, az = 0.f;
    for (int grp = lane; grp < groups; grp += 32) {
      const float4 f0 = __ldcs(val + 3 * grp), f1 = __ldcs(val + 3 * grp + 1), f2 = __ldcs(val + 3 * grp + 2);
      const float4 gv = __ldg(g4 + grp);
      ax = fmaf(gv.x, f0.x, ax); ay = fmaf(gv.x, f0.y, ay); az = fmaf(gv.x, f0.z, az);
      ax = fmaf(gv.y, f0.w, ax); ay = fmaf(gv.y, f1.x, ay); az = fmaf(gv.y, f1.y, az);
      ax = fmaf(gv.z, f1.z, ax); ay = fmaf(gv.z, f1.w, ay); az = fmaf(gv.z, f2.x, az);
      ax = fmaf(gv.w, f2.y, ax); ay = fmaf(gv.w, f2.z, ay); az = fmaf(gv.w, f2.w, az);
    }
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) {
      ax += __shfl_xor_sync(0xffffffffu, ax, m);
      ay += __shfl_xor_sync(0xffffffffu, ay, m);
      az += __shfl_xor_sync(0xffffffffu, az, m);
    }
    if (lane == 0) {
      atomicAdd(forces + (size_t)j * 3 + 0, -ax);
      atomicAdd(forces + (size_t)j * 3 + 1, -ay);
      atomicAdd(forces + (size_t)j * 3 + 2, -az);
    }
  }
}

int device_sm_count();

int contract_dense(const float* g, const int32_t* mol_off, int32_t n_mol, int64_t n_atoms, int d,
                   const float* dense, const int64_t* dense_off, float* forces, cudaStream_t st) {
  QMLL_CUDA_TRY(cudaMemsetAsync(forces, 0, (size_t)n_atoms * 3 * sizeof(float), st));
  if (n_mol == 0 || n_atoms == 0) return QMLL_OK;
  // enough blocks for ~8 per SM even with few molecules; rows of a molecule are split across blockIdx.y
  const int want = device_sm_count() * 32;
  int splits = (want + n_mol - 1) / n_mol;
  if (splits < 1) splits = 1;
  if (splits > 64) splits = 64;
  // blockIdx.x is limited to 2^31-1 and n_mol is an int32: fine
  dim3 grid((unsigned)n_mol, (unsigned)splits);
  contract_dense_kernel<<<grid, kCtrThreads, 0, st>>>(g, mol_off, d, dense, dense_off, forces, splits);
  QMLL_LAUNCH_CHECK("contract_dense_kernel");
  return QMLL_OK;
}

int contract_neighbor(const float* g, int64_t n_atoms, int d, int K, const int32_t* nbr_idx,
                      const float* nbr_val, float* forces, cudaStream_t st) {
  QMLL_CUDA_TRY(cudaMemsetAsync(forces, 0, (size_t)n_atoms * 3 * sizeof(float), st));
  const long long n_pairs = (long long)n_atoms * K;
  if (n_pairs == 0) return QMLL_OK;
  const long long warps_per_block = kCtrThreads / 32;
  long long blocks = (n_pairs + warps_per_block - 1) / warps_per_block;
  const long long cap = (long long)device_sm_count() * 8 * 16;  // grid-stride beyond ~16 waves
  if (blocks > cap) blocks = cap;
  contract_neighbor_kernel<<<(unsigned)blocks, kCtrThreads, 0, st>>>(g, n_pairs, d, K, nbr_idx, nbr_val, forces);
  QMLL_LAUNCH_CHECK("contract_neighbor_kernel");
  return QMLL_OK;
}

}  // namespace qmll
