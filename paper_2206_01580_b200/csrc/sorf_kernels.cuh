// sorf_kernels.cuh -- the fused SORF kernels (steps a1-a7 of SURVEY.md section 8):
//   sorf_forward_kernel      sign/FWHT chain -> cos -> per-molecule segmented sum -> Z              (eq. 20, 14, 15)
//   sorf_predict_kernel      chain -> sin/cos -> energies, transposed chain -> g = dE/dx -> fused contraction with the
//                            descriptor gradient -> forces                                           (L268, L137, L63)
//   sorf_force_rows_*_kernel JVP of the chain on descriptor-gradient columns -> G = -dZ/dr           (L137, eq. 17)
// Per-atom features never reach HBM in the forward and predict kernels, and neither does g.
#pragma once
#include <math.h>

#include "qmll_common.cuh"
#include "sorf_device.cuh"
#include "ptx_utils.cuh"

namespace qmll {

constexpr int kFwdThreads = 128;  // forward: 4 warps; smem accumulators: E * 128 * 4 B (64 KB at E = 128)
constexpr int kPredThreads = 256; // predict: 8 warps, one block per SM (the chain + accumulators want ~200 registers)
constexpr int kRowsMaxWarps = 10; // force rows: up to 10 warps (rows of one molecule) share one staged sin table

// ------------------------------------------------------------------------------------------------
// Forward (a1-a3).  Warp task = (atom chunk, stack group of SPW stacks).  The warp walks the atoms of its
// chunk; each lane runs the chain for its stack in registers, adds cos(.) into its private accumulator column
// in shared memory, and at every molecule boundary the warp writes the finished [SPW, d] slab of Z (scaled by
// sqrt(2/D)) with coalesced float4 stores (atomics only for molecules cut by a chunk border).
// If zs_out != NULL the per-atom sqrt(2/D) sin(.) is also written for the force-row kernel, as one contiguous
// block per (atom, stack group): zs[((a * n_sg + sg) * E4 + q) * 32 + lane] (float4).
// ------------------------------------------------------------------------------------------------
template <typename S, int NT>
__device__ __forceinline__ void flush_slab(float4* acc, int warp_tid0, int lane, float* __restrict__ dst_row,
                                           int sg, int n_s, float scale, bool atomic) {
  // acc[(j4 * NT) + tid]; slab of stack sl lives in lanes sl*P .. sl*P+P-1 of this warp
  __syncwarp();
#pragma unroll 1
  for (int sl = 0; sl < S::SPW; ++sl) {
    const int s = sg * S::SPW + sl;
    if (s >= n_s) break;
    float* dst = dst_row + (size_t)s * S::d;
    for (int q = lane; q < S::d / 4; q += kWarp) {
      const int m = 4 * q, p = m / S::E, j4 = (m % S::E) / 4;
      float4 a = acc[j4 * NT + warp_tid0 + sl * S::P + p];
      a.x *= scale; a.y *= scale; a.z *= scale; a.w *= scale;
      if (atomic) {
        atomicAdd(dst + m + 0, a.x); atomicAdd(dst + m + 1, a.y);
        atomicAdd(dst + m + 2, a.z); atomicAdd(dst + m + 3, a.w);
      } else {
        *reinterpret_cast<float4*>(dst + m) = a;
      }
    }
  }
  __syncwarp();
}

template <typename S, int NT>
__device__ __forceinline__ void zero_acc(float4* acc, int tid) {
#pragma unroll
  for (int q = 0; q < S::E4; ++q) acc[q * NT + tid] = make_float4(0.f, 0.f, 0.f, 0.f);
}

template <typename S, bool kWriteSin>
__global__ void __launch_bounds__(kFwdThreads, (S::E >= 128 ? 3 : 4))
sorf_forward_kernel(const float* __restrict__ x, const int32_t* __restrict__ elem,
                    const int32_t* __restrict__ mol_off, int n_atoms, int n_mol, int n_s, int T, float c,
                    float nrm, const uint32_t* __restrict__ sign_bits, const float* __restrict__ bias_t,
                    float* __restrict__ Z, float* __restrict__ zs_out, int chunk, int n_chunks, int n_sg) {
  extern __shared__ float4 acc[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const long long task = (long long)blockIdx.x * (kFwdThreads / kWarp) + warp;
  if (task >= (long long)n_chunks * n_sg) return;
  const int sg = (int)(task % n_sg), ch = (int)(task / n_sg);
  const int p = lane % S::P;

  const int a_begin = chunk_cut(mol_off, n_mol, n_atoms, ch, chunk);
  const int a_end = chunk_cut(mol_off, n_mol, n_atoms, ch + 1, chunk);
  if (a_begin >= a_end) return;

  zero_acc<S, kFwdThreads>(acc, tid);
  int mol = owner_molecule(mol_off, n_mol, a_begin);
  int mol_lo = __ldg(mol_off + mol), mol_hi = __ldg(mol_off + mol + 1);
  const float4* bias4 = reinterpret_cast<const float4*>(bias_t);
  const f32x2 c2 = pk(c, c);

#pragma unroll 1
  for (int a = a_begin; a < a_end; ++a) {
    if (a >= mol_hi) {  // molecule finished inside this task
      if (Z) flush_slab<S, kFwdThreads>(acc, warp * kWarp, lane, Z + (size_t)mol * (size_t)n_s * S::d, sg, n_s, nrm,
                                        mol_lo < a_begin);
      zero_acc<S, kFwdThreads>(acc, tid);
      do { ++mol; mol_hi = __ldg(mol_off + mol + 1); } while (a >= mol_hi);
      mol_lo = __ldg(mol_off + mol);
    }
    const int e = __ldg(elem + a);
    f32x2 v[S::E2];
    load_row<S>(v, x + (size_t)a * S::d, p);
    chain_forward<S>(v, sign_bits, e, T, n_sg, sg, lane);
    const float4* b4 = bias4 + ((size_t)e * n_sg + sg) * (S::E4 * kWarp) + lane;
    float4* zs4 = kWriteSin ? reinterpret_cast<float4*>(zs_out) + ((size_t)a * n_sg + sg) * (S::E4 * kWarp) + lane
                            : nullptr;
#pragma unroll
    for (int q = 0; q < S::E4; ++q) {
      const float4 b = __ldg(b4 + q * kWarp);
      float t0, t1, t2, t3;
      upk(fma2(v[2 * q], c2, pk(b.x, b.y)), t0, t1);       // u + b in radians; MUFU's own range reduction is
      upk(fma2(v[2 * q + 1], c2, pk(b.z, b.w)), t2, t3);   // as accurate as the fp32 rounding of u + b itself
      float4 ac = acc[q * kFwdThreads + tid];
      ac.x += __cosf(t0); ac.y += __cosf(t1); ac.z += __cosf(t2); ac.w += __cosf(t3);
      acc[q * kFwdThreads + tid] = ac;
      if (kWriteSin)
        zs4[(size_t)q * kWarp] = make_float4(nrm * __sinf(t0), nrm * __sinf(t1), nrm * __sinf(t2), nrm * __sinf(t3));
    }
  }
  if (Z) flush_slab<S, kFwdThreads>(acc, warp * kWarp, lane, Z + (size_t)mol * (size_t)n_s * S::d, sg, n_s, nrm,
                                    mol_lo < a_begin || mol_hi > a_end);
}

// ------------------------------------------------------------------------------------------------
// Predict / backward (a1, a4, a5, a6 fused).  Block = 8 warps, each warp owns one atom at a time and loops over
// all stack groups:   u -> (cos, sin) of the same argument;  energy += alpha_s * cos;  q = alpha_s * sin;
// transposed chain;  the per-lane results are summed over the stack groups in shared memory, then over the SPW
// stack lanes once per atom:  gbuf = c * sum_s W_{e,s}^T q_s = -dE/dx_I.  The warp then streams the atom's block of
// the descriptor gradient exactly once and adds  F[j, k] += sum_m gbuf[m] * dx_I[m]/dr_{j,k}  (F = -dE/dr, eq. 5/10)
// with one float atomic per (atom, column) -- the ALU-bound chain of some warps overlaps the HBM-bound gradient
// stream of others, and g never leaves the SM.  The block's warps step through the stack groups together
// (__syncthreads per group) so that the group's bias / alpha / sign tables stay resident in L1.
// energy_acc[mol] (double, pre-zeroed) receives one atomicAdd per atom.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
  return v;
}

struct GradView {          // qmll_grad flattened for the device
  int layout;              // QMLL_GRAD_NONE / DENSE / NEIGHBOR
  const float* dense;
  const int64_t* dense_off;
  const int32_t* nbr_idx;
  const float* nbr_val;
  int K;
};

// F[a0 + j, k] += sum_m gbuf[m] * dx[Il][m][3 j + k]   (dense layout, A12): lane = column, rows streamed 16 deep.
template <typename S>
__device__ __forceinline__ void contract_dense_atom(const float* __restrict__ gbuf, const float* __restrict__ blk,
                                                    int ncol, float* __restrict__ Fmol, int lane) {
  for (int c0 = 0; c0 < ncol; c0 += kWarp) {
    const int col = c0 + lane;
    const bool ok = col < ncol;
    const float* ptr = blk + (ok ? col : 0);
    float s0 = 0.f, s1 = 0.f;
#pragma unroll 1
    for (int m = 0; m < S::d; m += 16) {
      float a[16];
#pragma unroll
      for (int u = 0; u < 16; ++u) a[u] = __ldcs(ptr + (size_t)(m + u) * ncol);
#pragma unroll
      for (int u = 0; u < 16; u += 4) {
        const float4 g = *reinterpret_cast<const float4*>(gbuf + m + u);
        s0 = fmaf(g.x, a[u], s0); s1 = fmaf(g.y, a[u + 1], s1);
        s0 = fmaf(g.z, a[u + 2], s0); s1 = fmaf(g.w, a[u + 3], s1);
      }
    }
    if (ok) atomicAdd(Fmol + col, s0 + s1);
  }
}

// F[j, k] += sum_m gbuf[m] * val[q][m][k], j = nbr_idx[a, q]   (neighbour layout, A13; duplicates and self add,
// -1 = padding): each [d, 3] block is 3d contiguous floats; a lane takes 12 of them (4 values of m) per step.
template <typename S>
__device__ __forceinline__ void contract_neighbor_atom(const float* __restrict__ gbuf, const int32_t* __restrict__ idx,
                                                       const float* __restrict__ val, int K, float* __restrict__ F,
                                                       int lane) {
  constexpr int G = S::d / 4;                          // groups of 12 floats per block
  constexpr int GPL = (G + kWarp - 1) / kWarp;         // groups per lane
  const float4* g4 = reinterpret_cast<const float4*>(gbuf);
#pragma unroll 1
  for (int q = 0; q < K; ++q) {
    const int j = __ldg(idx + q);
    if (j < 0) continue;
    const float4* v4 = reinterpret_cast<const float4*>(val + (size_t)q * S::d * 3);
    float4 f[GPL][3];
#pragma unroll
    for (int t = 0; t < GPL; ++t) {
      const int grp = lane + kWarp * t;
      if (G % kWarp == 0 || grp < G) {
        f[t][0] = __ldcs(v4 + 3 * grp); f[t][1] = __ldcs(v4 + 3 * grp + 1); f[t][2] = __ldcs(v4 + 3 * grp + 2);
      } else {
        f[t][0] = f[t][1] = f[t][2] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
    }
    float ax = 0.f, ay = 0.f, az = 0.f;
#pragma unroll
    for (int t = 0; t < GPL; ++t) {
      const int grp = lane + kWarp * t;
      const float4 gv = (G % kWarp == 0 || grp < G) ? g4[grp] : make_float4(0.f, 0.f, 0.f, 0.f);
      const float4 f0 = f[t][0], f1 = f[t][1], f2 = f[t][2];
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
      atomicAdd(F + (size_t)j * 3 + 0, ax);
      atomicAdd(F + (size_t)j * 3 + 1, ay);
      atomicAdd(F + (size_t)j * 3 + 2, az);
    }
  }
}

template <typename S>
struct PredSmem {
  static constexpr int kWarps = kPredThreads / kWarp;
  static constexpr size_t kAccBytes = (size_t)S::E * kWarp * sizeof(float);       // per warp: [E4][32] float4
  static constexpr size_t kBytes = kWarps * (kAccBytes + S::d * sizeof(float));   // + gbuf[d] per warp
};

template <typename S, bool kNeedG>
__global__ void __launch_bounds__(kPredThreads, 1)
sorf_predict_kernel(const float* __restrict__ x, const int32_t* __restrict__ elem,
                    const int32_t* __restrict__ mol_off, int n_atoms, int n_mol, int n_s, int T, float c,
                    const uint32_t* __restrict__ sign_bits, const float* __restrict__ bias_t,
                    const float* __restrict__ alpha_s, GradView grad, float* __restrict__ forces,
                    double* __restrict__ energy_acc, int atoms_per_block, int n_sg) {
  extern __shared__ float4 smem4[];
  constexpr int kWarps = kPredThreads / kWarp;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  float4* acc = smem4 + warp * (S::E4 * kWarp);                                           // [E4][32]
  float* gbuf = reinterpret_cast<float*>(smem4 + kWarps * (S::E4 * kWarp)) + warp * S::d;  // [d]
  const int p = lane % S::P;
  const int a_block = blockIdx.x * atoms_per_block;
  const int a_stop = a_block + atoms_per_block < n_atoms ? a_block + atoms_per_block : n_atoms;
  const float4* bias4 = reinterpret_cast<const float4*>(bias_t);
  const float4* alpha4 = reinterpret_cast<const float4*>(alpha_s);
  const f32x2 c2 = pk(c, c);

#pragma unroll 1
  for (int a0 = a_block; a0 < a_stop; a0 += kWarps) {
    const int a = a0 + warp;
    const bool have = a < a_stop;
    const int e = have ? __ldg(elem + a) : 0;
    f32x2 epart2 = pk(0.f, 0.f);
    if (kNeedG && have) {
#pragma unroll
      for (int q = 0; q < S::E4; ++q) acc[q * kWarp + lane] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
#pragma unroll 1
    for (int sg = 0; sg < n_sg; ++sg) {
      __syncthreads();  // the block's warps stay on the same stack group: its tables are L1-resident
      if (!have) continue;
      f32x2 v[S::E2];
      load_row<S>(v, x + (size_t)a * S::d, p);
      const float4* b4 = bias4 + ((size_t)e * n_sg + sg) * (S::E4 * kWarp) + lane;
      const float4* al4 = alpha4 + (size_t)sg * (S::E4 * kWarp) + lane;
      // Forward chain, sin/cos, transposed chain as ONE loop over 2T phases so that the unrolled butterfly and
      // sign-flip code exist once (instruction cache).  Phase i < T: S_i then H.  Phase T: u -> (energy, q), then H
      // (with all-plus signs).  Phase T < i < 2T: S_{2T-i} then H.  The last sign flip S_0 is folded into the
      // accumulation below.   [ (H S_{T-1} ... H S_0) x ;  S_0 H S_1 H ... S_{T-1} H q ]
      const int n_phase = kNeedG ? 2 * T : T + 1;
#pragma unroll 1
      for (int i = 0; i < n_phase; ++i) {
        uint32_t w[S::EW];
        if (i == T) {
#pragma unroll
          for (int q = 0; q < S::E4; ++q) {
            const float4 b = __ldg(b4 + q * kWarp);
            const float4 al = __ldg(al4 + q * kWarp);   // zero for the idle lanes of the last stack group
            float t0, t1, t2, t3;
            upk(fma2(v[2 * q], c2, pk(b.x, b.y)), t0, t1);
            upk(fma2(v[2 * q + 1], c2, pk(b.z, b.w)), t2, t3);
            const f32x2 al01 = pk(al.x, al.y), al23 = pk(al.z, al.w);
            epart2 = fma2(al01, pk(__cosf(t0), __cosf(t1)), epart2);
            epart2 = fma2(al23, pk(__cosf(t2), __cosf(t3)), epart2);
            if (kNeedG) {
              v[2 * q] = mul2(al01, pk(__sinf(t0), __sinf(t1)));
              v[2 * q + 1] = mul2(al23, pk(__sinf(t2), __sinf(t3)));
            }
          }
          if (!kNeedG) break;
#pragma unroll
          for (int k = 0; k < S::EW; ++k) w[k] = 0u;
        } else {
          const int t = i < T ? i : 2 * T - i;
          load_sign_words<S>(w, sign_bits, e, t, T, n_sg, sg, lane);
        }
        sign_fwht<S, true>(v, w, p);
      }
      if (kNeedG) {
        uint32_t w[S::EW];
        load_sign_words<S>(w, sign_bits, e, 0, T, n_sg, sg, lane);
#pragma unroll
        for (int q = 0; q < S::E4; ++q) {
          float t0, t1, t2, t3;
          upk(v[2 * q], t0, t1);
          upk(v[2 * q + 1], t2, t3);
          const int j = 4 * q;
          const uint32_t ws = w[j >> 5];
          t0 = __uint_as_float(__float_as_uint(t0) ^ ((ws << (31 - (j & 31))) & 0x80000000u));
          t1 = __uint_as_float(__float_as_uint(t1) ^ ((ws << (30 - (j & 31))) & 0x80000000u));
          t2 = __uint_as_float(__float_as_uint(t2) ^ ((ws << (29 - (j & 31))) & 0x80000000u));
          t3 = __uint_as_float(__float_as_uint(t3) ^ ((ws << (28 - (j & 31))) & 0x80000000u));
          float4 ac = acc[q * kWarp + lane];
          ac.x += t0; ac.y += t1; ac.z += t2; ac.w += t3;
          acc[q * kWarp + lane] = ac;
        }
      }
    }
    if (!have) continue;
    int M = 0, m_lo = 0, n = 0;
    if (energy_acc != nullptr || (kNeedG && grad.layout == QMLL_GRAD_DENSE)) {
      M = owner_molecule(mol_off, n_mol, a);
      m_lo = __ldg(mol_off + M);
      n = __ldg(mol_off + M + 1) - m_lo;
    }
    if (energy_acc != nullptr) {
      float e0, e1;
      upk(epart2, e0, e1);
      const float tot = warp_sum(e0 + e1);
      if (lane == 0) atomicAdd(energy_acc + M, (double)tot);
    }
    if (kNeedG) {
      // sum the per-lane accumulators over the SPW stack lanes: item (q, pp) -> gbuf[pp*E + 4q .. +3]
      __syncwarp();
#pragma unroll 1
      for (int item = lane; item < S::E4 * S::P; item += kWarp) {
        const int q = item / S::P, pp = item % S::P;
        float4 s4 = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 4
        for (int i = 0; i < S::SPW; ++i) {
          const int sl2 = (i + lane) % S::SPW;   // rotated start: the lanes of a warp hit different banks
          const float4 t = acc[q * kWarp + sl2 * S::P + pp];
          s4.x += t.x; s4.y += t.y; s4.z += t.z; s4.w += t.w;
        }
        s4.x *= c; s4.y *= c; s4.z *= c; s4.w *= c;
        *reinterpret_cast<float4*>(gbuf + pp * S::E + 4 * q) = s4;
      }
      __syncwarp();
      if (grad.layout == QMLL_GRAD_DENSE) {
        const float* blk = grad.dense + __ldg(grad.dense_off + M) + (size_t)(a - m_lo) * S::d * 3 * n;
        contract_dense_atom<S>(gbuf, blk, 3 * n, forces + (size_t)m_lo * 3, lane);
      } else {
        contract_neighbor_atom<S>(gbuf, grad.nbr_idx + (size_t)a * grad.K,
                                  grad.nbr_val + (size_t)a * grad.K * S::d * 3, grad.K, forces, lane);
      }
      __syncwarp();
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Force rows (a7), dense gradient.  Block task = (a group of up to W rows r = 3*j + k of ONE molecule, stack group);
// warp w owns one row.  All warps loop together over the atoms I of the molecule: the gradient column
// dx_I[:, j, k] of the warp's row goes through the same chain as x (JVP of a linear map = the map itself), is
// weighted by sqrt(2/D) sin(u_I + b) of that (atom, stack group) and summed over I in the warp's shared-memory
// accumulators; the finished [SPW, d] slab of G row r is then written once.
//   G[r, l] = c * sum_I zs_I[l] * (H S_T ... H S_1 dx_I[:, j, k])[l]
// The sin table of (I, stack group) -- E*128 bytes, written by the forward kernel -- is staged ONCE per block and
// atom by a TMA bulk copy into a 2-slot ring (full / empty mbarriers) and read by all W warps, so it crosses L2
// once per W rows; every warp stages its own gradient column the same way (2-slot ring, 1-D bulk copies of the
// column made contiguous by transpose_dense_kernel).
// ------------------------------------------------------------------------------------------------
template <typename S>
struct RowsSmem {
  static constexpr int kSlice = S::E + 4;                 // floats per lane slice (+16 B: no bank conflicts for P > 1)
  static constexpr int kColFloats = S::P * kSlice;        // one staged column
  static constexpr size_t kAccBytes = (size_t)S::E * kWarp * sizeof(float);   // per warp [E4][32] float4
  static constexpr size_t kZsBytes = kAccBytes;                               // one (atom, stack group) sin table
  static size_t bytes(int W) {
    return (size_t)W * kAccBytes + 2 * kZsBytes + (size_t)W * 2 * kColFloats * sizeof(float) +
           (size_t)(4 + 2 * W) * sizeof(uint64_t);
  }
};

template <typename S>
__global__ void __launch_bounds__(kRowsMaxWarps * kWarp, 1)
sorf_force_rows_dense_kernel(const int32_t* __restrict__ elem, const int32_t* __restrict__ mol_off, int n_atoms,
                             int n_mol, int n_s, int T, float c, const uint32_t* __restrict__ sign_bits,
                             const float* __restrict__ zs, const float* __restrict__ gt,
                             const int64_t* __restrict__ dense_off, const int32_t* __restrict__ grp_off,
                             float* __restrict__ G, int n_sg, int W) {
  extern __shared__ float4 smem4[];
  using RS = RowsSmem<S>;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  float4* acc = smem4 + warp * (S::E4 * kWarp);
  float4* zsbuf = smem4 + W * (S::E4 * kWarp);                       // [2][E4][32]
  float* colbuf = reinterpret_cast<float*>(zsbuf + 2 * (S::E4 * kWarp)) + warp * 2 * RS::kColFloats;
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<float*>(zsbuf + 2 * (S::E4 * kWarp)) +
                                               W * 2 * RS::kColFloats);
  uint64_t* zs_full = bars;          // [2]
  uint64_t* zs_empty = bars + 2;     // [2]
  uint64_t* col_bar = bars + 4 + 2 * warp;  // [2] per warp

  // block -> (molecule M, row group rg, stack group sg); grp_off[M] = number of row groups before molecule M
  const int sg = blockIdx.x % n_sg;
  const int g = blockIdx.x / n_sg;
  if (g >= __ldg(grp_off + n_mol)) return;
  int lo = 0, hi = n_mol - 1;
  while (lo < hi) { const int mid = (lo + hi) >> 1; if (__ldg(grp_off + mid + 1) > g) hi = mid; else lo = mid + 1; }
  const int M = lo, rg = g - __ldg(grp_off + M), n_grp = __ldg(grp_off + M + 1) - __ldg(grp_off + M);
  const int a0 = __ldg(mol_off + M), n = __ldg(mol_off + M + 1) - a0;
  const int r_lo = (int)((long long)3 * n * rg / n_grp), r_hi = (int)((long long)3 * n * (rg + 1) / n_grp);
  const int n_rows = r_hi - r_lo;    // <= W active warps
  const int p = lane % S::P;

  if (tid == 0) {
    mbar_init(&zs_full[0], 1); mbar_init(&zs_full[1], 1);
    mbar_init(&zs_empty[0], n_rows); mbar_init(&zs_empty[1], n_rows);
    for (int w = 0; w < W; ++w) { mbar_init(bars + 4 + 2 * w, 1); mbar_init(bars + 5 + 2 * w, 1); }
    fence_mbarrier_init();
  }
  __syncthreads();
  if (warp >= n_rows) return;

  const int rl = r_lo + warp;                     // local row 3*jl + k of molecule M
  const long long r = (long long)3 * a0 + rl;     // global row of G
  // column (I, jl, k) of molecule M: d contiguous floats of gt; consecutive I are 3*n*d floats apart
  const float* col0 = gt + __ldg(dense_off + M) + (size_t)rl * S::d;
  const size_t istride = (size_t)3 * n * S::d;
  const float* zs_src = zs + ((size_t)a0 * n_sg + sg) * (S::E * kWarp);   // + I * n_sg * E*32 floats
  const size_t zs_stride = (size_t)n_sg * S::E * kWarp;

  auto stage_col = [&](int I) {  // lane 0 of each warp
    uint64_t* bar = &col_bar[I & 1];
    float* dst = colbuf + (I & 1) * RS::kColFloats;
    mbar_expect_tx(bar, S::d * sizeof(float));
#pragma unroll
    for (int pp = 0; pp < S::P; ++pp)
      bulk_copy_g2s(dst + pp * RS::kSlice, col0 + (size_t)I * istride + pp * S::E, S::E * sizeof(float), bar);
  };
  auto stage_zs = [&](int I) {   // thread 0 of the block
    const int slot = I & 1, use = I >> 1;
    if (use > 0) mbar_wait(&zs_empty[slot], (uint32_t)((use - 1) & 1));   // all warps are done with the previous tenant
    mbar_expect_tx(&zs_full[slot], (uint32_t)RS::kZsBytes);
    bulk_copy_g2s(zsbuf + slot * (S::E4 * kWarp), zs_src + (size_t)I * zs_stride, (uint32_t)RS::kZsBytes,
                  &zs_full[slot]);
  };
  if (tid == 0) stage_zs(0);
  if (lane == 0) stage_col(0);

#pragma unroll
  for (int q = 0; q < S::E4; ++q) acc[q * kWarp + lane] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 1
  for (int I = 0; I < n; ++I) {
    if (I + 1 < n) {
      if (tid == 0) stage_zs(I + 1);
      if (lane == 0) stage_col(I + 1);   // slot (I+1)&1 was last read in iteration I-1 (warp-synced below)
    }
    const int e = __ldg(elem + a0 + I);
    mbar_wait(&col_bar[I & 1], (uint32_t)((I >> 1) & 1));
    f32x2 v[S::E2];
    load_row<S>(v, colbuf + (I & 1) * RS::kColFloats + p * 4, p);   // slices are kSlice = E + 4 floats apart
    __syncwarp();
    chain_forward<S>(v, sign_bits, e, T, n_sg, sg, lane);
    mbar_wait(&zs_full[I & 1], (uint32_t)((I >> 1) & 1));
    const float4* z4 = zsbuf + (I & 1) * (S::E4 * kWarp) + lane;
#pragma unroll
    for (int q = 0; q < S::E4; ++q) {
      const float4 z = z4[q * kWarp];
      float4 ac = acc[q * kWarp + lane];
      f32x2 a01 = fma2(pk(z.x, z.y), v[2 * q], pk(ac.x, ac.y));
      f32x2 a23 = fma2(pk(z.z, z.w), v[2 * q + 1], pk(ac.z, ac.w));
      upk(a01, ac.x, ac.y);
      upk(a23, ac.z, ac.w);
      acc[q * kWarp + lane] = ac;
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&zs_empty[I & 1]);
  }
  flush_slab<S, kWarp>(acc, 0, lane, G + (size_t)r * (size_t)n_s * S::d, sg, n_s, c, false);
}

// Number of row groups of every molecule: grp_off[M] = sum_{M' < M} ceil(3 n_M' / W)  (one block, serial scan over
// chunks of 1024 molecules; n_mol is at most a few hundred thousand).
static __global__ void __launch_bounds__(1024)
row_group_offsets_kernel(const int32_t* __restrict__ mol_off, int n_mol, int W, int32_t* __restrict__ grp_off) {
  __shared__ int part[1024];
  __shared__ int carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int base = 0; base < n_mol; base += 1024) {
    const int M = base + threadIdx.x;
    const int cnt = M < n_mol ? (3 * (__ldg(mol_off + M + 1) - __ldg(mol_off + M)) + W - 1) / W : 0;
    part[threadIdx.x] = cnt;
    __syncthreads();
    for (int off = 1; off < 1024; off <<= 1) {   // inclusive scan
      const int t = threadIdx.x >= off ? part[threadIdx.x - off] : 0;
      __syncthreads();
      part[threadIdx.x] += t;
      __syncthreads();
    }
    if (M < n_mol) grp_off[M] = carry + part[threadIdx.x] - cnt;
    __syncthreads();
    if (threadIdx.x == 1023) carry += part[1023];
    __syncthreads();
  }
  if (threadIdx.x == 0) grp_off[n_mol] = carry;
}

// Force rows, neighbour-sparse gradient (A13): rows of different atoms collide, so contributions are added
// with atomics into a pre-zeroed G.  Warp task = (atom I, neighbour slot q, stack group), 3 columns each.
template <typename S>
__global__ void __launch_bounds__(kFwdThreads, (S::E >= 128 ? 3 : 4))
sorf_force_rows_neighbor_kernel(const int32_t* __restrict__ elem, int n_atoms, int n_s, int T, float c,
                                const uint32_t* __restrict__ sign_bits, const float* __restrict__ zs,
                                const int32_t* __restrict__ nbr_idx, const float* __restrict__ nbr_val, int K,
                                float* __restrict__ G, int n_sg) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const long long task = (long long)blockIdx.x * (kFwdThreads / kWarp) + warp;
  if (task >= (long long)n_atoms * K * n_sg) return;
  const int sg = (int)(task % n_sg);
  const long long iq = task / n_sg;
  const int I = (int)(iq / K);
  const int jg = __ldg(nbr_idx + iq);
  if (jg < 0) return;
  const int p = lane % S::P, sl = lane / S::P;
  const int s_raw = sg * S::SPW + sl;
  const bool valid = s_raw < n_s;
  const int e = __ldg(elem + I);
  const float4* z4 = reinterpret_cast<const float4*>(zs) + ((size_t)I * n_sg + sg) * (S::E4 * kWarp) + lane;
  const float* val = nbr_val + (size_t)iq * S::d * 3;
#pragma unroll 1
  for (int k = 0; k < 3; ++k) {
    f32x2 v[S::E2];
#pragma unroll
    for (int j = 0; j < S::E2; ++j)
      v[j] = pk(__ldg(val + (size_t)(p * S::E + 2 * j) * 3 + k), __ldg(val + (size_t)(p * S::E + 2 * j + 1) * 3 + k));
    chain_forward<S>(v, sign_bits, e, T, n_sg, sg, lane);
    if (valid) {
      float* dst = G + ((size_t)jg * 3 + k) * (size_t)n_s * S::d + (size_t)s_raw * S::d + p * S::E;
#pragma unroll
      for (int q = 0; q < S::E4; ++q) {
        const float4 z = __ldg(z4 + (size_t)q * kWarp);
        float t0, t1, t2, t3;
        upk(v[2 * q], t0, t1);
        upk(v[2 * q + 1], t2, t3);
        atomicAdd(dst + 4 * q + 0, c * z.x * t0); atomicAdd(dst + 4 * q + 1, c * z.y * t1);
        atomicAdd(dst + 4 * q + 2, c * z.z * t2); atomicAdd(dst + 4 * q + 3, c * z.w * t3);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Host-side launchers for one shape S.
// ------------------------------------------------------------------------------------------------
int device_sm_count();

static inline int clampi(long long v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : (int)v); }

template <typename S>
struct SorfLaunch {
  static constexpr int kWarpsPerBlock = kFwdThreads / kWarp;
  static constexpr size_t kAccBytes = (size_t)S::E * kFwdThreads * sizeof(float);

  static float c_of(const qmll_sorf_params* p) {
    return (float)(sqrt((double)p->d) / (double)p->sigma * pow((double)p->d, -0.5 * p->n_transform));
  }
  static int warp_slots() { return device_sm_count() * kWarpsPerBlock * (S::E >= 128 ? 3 : 4); }

  static int forward(const SorfProblem& pr, const SorfTables& t, float* Z, float* zs_out, cudaStream_t st) {
    const qmll_sorf_params* p = pr.p;
    const int n_s = p->D / p->d, n_sg = (n_s + S::SPW - 1) / S::SPW;
    const int n_atoms = (int)pr.n_atoms;
    if (Z) QMLL_CUDA_TRY(cudaMemsetAsync(Z, 0, (size_t)pr.n_mol * p->D * sizeof(float), st));
    if (n_atoms == 0 || pr.n_mol == 0) return QMLL_OK;
    const int chunk = clampi((long long)n_atoms * n_sg / (4LL * warp_slots()), 4, 32);
    const int n_chunks = (n_atoms + chunk - 1) / chunk;
    const long long tasks = (long long)n_chunks * n_sg;
    const unsigned grid = (unsigned)((tasks + kWarpsPerBlock - 1) / kWarpsPerBlock);
    const float nrm = (float)sqrt(2.0 / (double)p->D);
    auto kern = zs_out ? sorf_forward_kernel<S, true> : sorf_forward_kernel<S, false>;
    QMLL_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kAccBytes));
    kern<<<grid, kFwdThreads, kAccBytes, st>>>(pr.x, pr.elem, pr.mol_off, n_atoms, pr.n_mol, n_s,
                                               p->n_transform, c_of(p), nrm, t.sign_bits, t.bias_t, Z, zs_out,
                                               chunk, n_chunks, n_sg);
    QMLL_LAUNCH_CHECK("sorf_forward_kernel");
    return QMLL_OK;
  }

  // energies (energy_acc != NULL) and / or forces (forces != NULL, pre-zeroed, with gv)
  static int predict(const SorfProblem& pr, const SorfTables& t, const GradView& gv, float* forces,
                     double* energy_acc, cudaStream_t st) {
    const qmll_sorf_params* p = pr.p;
    const int n_s = p->D / p->d, n_sg = (n_s + S::SPW - 1) / S::SPW;
    const int n_atoms = (int)pr.n_atoms;
    if (n_atoms == 0 || pr.n_mol == 0) return QMLL_OK;
    constexpr int kWarps = kPredThreads / kWarp;
    const int n_sm = device_sm_count();
    int apb = (n_atoms + n_sm - 1) / n_sm;
    apb = (apb + kWarps - 1) / kWarps * kWarps;
    const unsigned grid = (unsigned)((n_atoms + apb - 1) / apb);
    auto kern = forces ? sorf_predict_kernel<S, true> : sorf_predict_kernel<S, false>;
    const size_t smem = PredSmem<S>::kBytes;
    QMLL_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<grid, kPredThreads, smem, st>>>(pr.x, pr.elem, pr.mol_off, n_atoms, pr.n_mol, n_s, p->n_transform,
                                           c_of(p), t.sign_bits, t.bias_t, t.alpha_s, gv, forces, energy_acc, apb,
                                           n_sg);
    QMLL_LAUNCH_CHECK("sorf_predict_kernel");
    return QMLL_OK;
  }

  // rows-per-block W: as many as shared memory and registers allow, then the value that wastes the fewest warps
  // for molecules of the average size (exact when all molecules have the same number of atoms)
  static int rows_per_block(long long n_atoms, int n_mol) {
    int w_max = kRowsMaxWarps;
    while (w_max > 1 && RowsSmem<S>::bytes(w_max) > 220 * 1024) --w_max;
    const long long rows = n_mol > 0 ? (3 * n_atoms + n_mol - 1) / n_mol : 3;
    int best = w_max;
    double best_eff = 0.0;
    for (int w = w_max; w >= (w_max + 1) / 2; --w) {
      const double eff = (double)rows / (double)(((rows + w - 1) / w) * w);
      if (eff > best_eff + 1e-9) { best_eff = eff; best = w; }
    }
    return best;
  }

  static int force_rows_dense(const SorfProblem& pr, const SorfTables& t, const float* zs, const float* dense_t,
                              const int64_t* dense_off, int32_t* grp_off, float* G, cudaStream_t st) {
    const qmll_sorf_params* p = pr.p;
    const int n_s = p->D / p->d, n_sg = (n_s + S::SPW - 1) / S::SPW;
    const long long n_atoms = pr.n_atoms;
    if (n_atoms == 0) return QMLL_OK;
    const int W = rows_per_block(n_atoms, pr.n_mol);
    row_group_offsets_kernel<<<1, 1024, 0, st>>>(pr.mol_off, pr.n_mol, W, grp_off);
    QMLL_LAUNCH_CHECK("row_group_offsets_kernel");
    const long long groups_max = (3 * n_atoms + W - 1) / W + pr.n_mol;   // >= sum_M ceil(3 n_M / W)
    const long long grid = groups_max * n_sg;
    if (grid > 0x7fffffffLL) return QMLL_ERR_UNSUPPORTED;
    auto kern = sorf_force_rows_dense_kernel<S>;
    const size_t smem = RowsSmem<S>::bytes(W);
    QMLL_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<(unsigned)grid, W * kWarp, smem, st>>>(pr.elem, pr.mol_off, (int)n_atoms, pr.n_mol, n_s, p->n_transform,
                                                  c_of(p), t.sign_bits, zs, dense_t, dense_off, grp_off, G, n_sg, W);
    QMLL_LAUNCH_CHECK("sorf_force_rows_dense_kernel");
    return QMLL_OK;
  }

  static int force_rows_neighbor(const SorfProblem& pr, const SorfTables& t, const float* zs,
                                 const int32_t* nbr_idx, const float* nbr_val, int K, float* G,
                                 cudaStream_t st) {
    const qmll_sorf_params* p = pr.p;
    const int n_s = p->D / p->d, n_sg = (n_s + S::SPW - 1) / S::SPW;
    const int n_atoms = (int)pr.n_atoms;
    QMLL_CUDA_TRY(cudaMemsetAsync(G, 0, (size_t)3 * n_atoms * p->D * sizeof(float), st));
    if (n_atoms == 0 || K == 0) return QMLL_OK;
    const long long tasks = (long long)n_atoms * K * n_sg;
    const long long grid = (tasks + kWarpsPerBlock - 1) / kWarpsPerBlock;
    if (grid > 0x7fffffffLL) return QMLL_ERR_UNSUPPORTED;
    sorf_force_rows_neighbor_kernel<S><<<(unsigned)grid, kFwdThreads, 0, st>>>(
        pr.elem, n_atoms, n_s, p->n_transform, c_of(p), t.sign_bits, zs, nbr_idx, nbr_val, K, G, n_sg);
    QMLL_LAUNCH_CHECK("sorf_force_rows_neighbor_kernel");
    return QMLL_OK;
  }
};

// One translation unit per descriptor length instantiates these (sorf_d*.cu) so they compile in parallel.
#define QMLL_DECLARE_SORF_SHAPE(TAG)                                                                          \
  int sorf_forward_##TAG(const SorfProblem&, const SorfTables&, float*, float*, cudaStream_t);                 \
  int sorf_predict_##TAG(const SorfProblem&, const SorfTables&, const GradView&, float*, double*, cudaStream_t); \
  int sorf_force_rows_dense_##TAG(const SorfProblem&, const SorfTables&, const float*, const float*,           \
                                  const int64_t*, int32_t*, float*, cudaStream_t);                             \
  int sorf_force_rows_neighbor_##TAG(const SorfProblem&, const SorfTables&, const float*, const int32_t*,      \
                                     const float*, int, float*, cudaStream_t);

#define QMLL_DEFINE_SORF_SHAPE_D(TAG, D_) QMLL_DEFINE_SORF_SHAPE(TAG, shape_E(D_), shape_P(D_))
#define QMLL_DEFINE_SORF_SHAPE(TAG, E_, P_)                                                                   \
  int sorf_forward_##TAG(const SorfProblem& pr, const SorfTables& t, float* Z, float* zs, cudaStream_t st) {   \
    return SorfLaunch<Shape<E_, P_>>::forward(pr, t, Z, zs, st);                                               \
  }                                                                                                            \
  int sorf_predict_##TAG(const SorfProblem& pr, const SorfTables& t, const GradView& gv, float* f, double* en, \
                         cudaStream_t st) {                                                                    \
    return SorfLaunch<Shape<E_, P_>>::predict(pr, t, gv, f, en, st);                                           \
  }                                                                                                            \
  int sorf_force_rows_dense_##TAG(const SorfProblem& pr, const SorfTables& t, const float* zs,                 \
                                  const float* dense, const int64_t* off, int32_t* grp, float* G,              \
                                  cudaStream_t st) {                                                           \
    return SorfLaunch<Shape<E_, P_>>::force_rows_dense(pr, t, zs, dense, off, grp, G, st);                     \
  }                                                                                                            \
  int sorf_force_rows_neighbor_##TAG(const SorfProblem& pr, const SorfTables& t, const float* zs,              \
                                     const int32_t* idx, const float* val, int K, float* G, cudaStream_t st) { \
    return SorfLaunch<Shape<E_, P_>>::force_rows_neighbor(pr, t, zs, idx, val, K, G, st);                      \
  }

QMLL_DECLARE_SORF_SHAPE(d16)
QMLL_DECLARE_SORF_SHAPE(d32)
QMLL_DECLARE_SORF_SHAPE(d64)
QMLL_DECLARE_SORF_SHAPE(d128)
QMLL_DECLARE_SORF_SHAPE(d256)
QMLL_DECLARE_SORF_SHAPE(d512)
QMLL_DECLARE_SORF_SHAPE(d1024)

}  // namespace qmll
