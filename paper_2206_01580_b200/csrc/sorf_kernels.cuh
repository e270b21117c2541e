// sorf_kernels.cuh -- the fused SORF kernels (steps a1-a5, a7 of SURVEY.md section 8):
//   sorf_forward_kernel      sign/FWHT chain -> cos -> per-molecule segmented sum -> Z   (eq. 20, 14, 15)
//   sorf_backward_kernel     chain -> sin/cos -> energies, transposed chain -> g = dE/dx  (L268, L137)
//   sorf_force_rows_kernel   JVP of the chain on descriptor-gradient columns -> G = -dZ/dr (L137, eq. 17)
// plus the tiny table-packing kernels that put signs / bias / alpha into lane-major order.
// Per-atom features never reach HBM in the forward and backward kernels.
#pragma once
#include <math.h>

#include "qmll_common.cuh"
#include "sorf_device.cuh"
#include "ptx_utils.cuh"

namespace qmll {

constexpr int kFwdThreads = 128;  // 4 warps; smem accumulators: E * 128 * 4 B (64 KB at E = 128)
constexpr float kTwoPi = 6.283185307179586f;

// ------------------------------------------------------------------------------------------------
// Forward (a1-a3).  Warp task = (atom chunk, stack group of SPW stacks).  The warp walks the atoms of its
// chunk; each lane runs the chain for its stack in registers, adds sqrt(2/D) cos(.) into its private
// accumulator column in shared memory, and at every molecule boundary the warp writes the finished
// [SPW, d] slab of Z with coalesced float4 stores (atomics only for molecules cut by a chunk border).
// If zs_out != NULL the per-atom sqrt(2/D) sin(.) is also written (lane-major) for the force-row kernel.
// ------------------------------------------------------------------------------------------------
template <typename S>
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
      float4 a = acc[j4 * kFwdThreads + warp_tid0 + sl * S::P + p];
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

template <typename S>
__device__ __forceinline__ void zero_acc(float4* acc, int tid) {
#pragma unroll
  for (int q = 0; q < S::E4; ++q) acc[q * kFwdThreads + tid] = make_float4(0.f, 0.f, 0.f, 0.f);
}

template <typename S, bool kWriteSin>
__global__ void __launch_bounds__(kFwdThreads, (S::E >= 128 ? 3 : 4))
sorf_forward_kernel(const float* __restrict__ x, const int32_t* __restrict__ elem,
                    const int32_t* __restrict__ mol_off, int n_atoms, int n_mol, int n_s, int T, float c_rev,
                    float nrm, const uint32_t* __restrict__ sign_bits, const float* __restrict__ bias_rev,
                    float* __restrict__ Z, float* __restrict__ zs_out, int chunk, int n_chunks, int n_sg) {
  extern __shared__ float4 acc[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const long long task = (long long)blockIdx.x * (kFwdThreads / kWarp) + warp;
  if (task >= (long long)n_chunks * n_sg) return;
  const int sg = (int)(task % n_sg), c = (int)(task / n_sg);
  const int p = lane % S::P, sl = lane / S::P;
  const int n_gl = n_s * S::P;
  const int s_raw = sg * S::SPW + sl;
  const int s = s_raw < n_s ? s_raw : n_s - 1;  // clamp idle lanes onto a valid stack (their results are dropped)
  const int gl = s * S::P + p;

  const int a_begin = chunk_cut(mol_off, n_mol, n_atoms, c, chunk);
  const int a_end = chunk_cut(mol_off, n_mol, n_atoms, c + 1, chunk);
  if (a_begin >= a_end) return;

  zero_acc<S>(acc, tid);
  float4* xb = acc + S::E4 * kFwdThreads + warp * kXchgFloat4PerWarp;  // cross-lane scratch (P > 1 only)
  int mol = owner_molecule(mol_off, n_mol, a_begin);
  int mol_lo = __ldg(mol_off + mol), mol_hi = __ldg(mol_off + mol + 1);
  const float4* bias4 = reinterpret_cast<const float4*>(bias_rev);

#pragma unroll 1
  for (int a = a_begin; a < a_end; ++a) {
    if (a >= mol_hi) {  // molecule finished inside this task
      if (Z) flush_slab<S>(acc, warp * kWarp, lane, Z + (size_t)mol * (size_t)n_s * S::d, sg, n_s, nrm,
                           mol_lo < a_begin);
      zero_acc<S>(acc, tid);
      do { ++mol; mol_hi = __ldg(mol_off + mol + 1); } while (a >= mol_hi);
      mol_lo = __ldg(mol_off + mol);
    }
    const int e = __ldg(elem + a);
    float v[S::E];
    load_row<S>(v, x + (size_t)a * S::d, p);
    chain_forward<S>(v, sign_bits, e, T, n_gl, gl, p, xb, lane);
    const float4* b4 = bias4 + (size_t)e * S::E4 * n_gl + gl;
    float4* zs4 = kWriteSin ? reinterpret_cast<float4*>(zs_out) + (size_t)a * S::E4 * n_gl + gl : nullptr;
#pragma unroll
    for (int q = 0; q < S::E4; ++q) {
      const float4 b = __ldg(b4 + (size_t)q * n_gl);
      const float f0 = frac_rev(fmaf(v[4 * q + 0], c_rev, b.x));
      const float f1 = frac_rev(fmaf(v[4 * q + 1], c_rev, b.y));
      const float f2 = frac_rev(fmaf(v[4 * q + 2], c_rev, b.z));
      const float f3 = frac_rev(fmaf(v[4 * q + 3], c_rev, b.w));
      float4 ac = acc[q * kFwdThreads + tid];
      ac.x += cos_rev(f0); ac.y += cos_rev(f1); ac.z += cos_rev(f2); ac.w += cos_rev(f3);
      acc[q * kFwdThreads + tid] = ac;
      if (kWriteSin) {
        if (s_raw < n_s)
          zs4[(size_t)q * n_gl] = make_float4(nrm * sin_rev(f0), nrm * sin_rev(f1), nrm * sin_rev(f2),
                                              nrm * sin_rev(f3));
      }
    }
  }
  if (Z) flush_slab<S>(acc, warp * kWarp, lane, Z + (size_t)mol * (size_t)n_s * S::d, sg, n_s, nrm,
                       mol_lo < a_begin || mol_hi > a_end);
}

// ------------------------------------------------------------------------------------------------
// Backward (a1, a4, a5).  Warp task = atom chunk; the warp loops over all stack groups of an atom so that
// g_I = c * sum_s W_{e,s}^T q_s is finished in registers and stored once (no atomics on g):
//   u -> (cos, sin) of the same argument;  energy += alpha_s * cos;  q = -alpha_s * sin;
//   transposed chain;  reduce-scatter over the SPW stack lanes (shuffles), accumulate over stack groups.
// energy_acc[mol] (double, pre-zeroed) receives one atomicAdd per (task, molecule).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float select_f32(bool c, float a, float b) {
  float r;
  asm("{\n.reg .pred p;\nsetp.ne.u32 p, %3, 0;\nselp.f32 %0, %1, %2, p;\n}" : "=f"(r) : "f"(a), "f"(b), "r"((unsigned)c));
  return r;
}

template <typename S>
struct StackReduce {
  static constexpr bool kScatter = (S::E >= S::SPW);
  static constexpr int R = kScatter ? S::E / S::SPW : S::E;  // values a lane ends up owning
  static constexpr int kLogSPW = ilog2(S::SPW);
  // One halving step: lanes whose bit `mask` is clear keep the lower half of the live elements and receive the
  // partner's lower half; the others keep / receive the upper half.  K is a template parameter so that every
  // register index is a compile-time constant (a runtime `half` sends v[] to local memory).
  template <int K>
  __device__ static __forceinline__ void step(float (&v)[S::E], int lane, int& jbase) {
    if constexpr (K < kLogSPW) {
      constexpr int mask = S::P << K;
      constexpr int half = S::E >> (K + 1);
      const bool up = (lane & mask) != 0;
#pragma unroll
      for (int i = 0; i < half; ++i) {
        const float send = select_f32(up, v[i], v[i + half]);
        const float keep = select_f32(up, v[i + half], v[i]);
        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, mask);
      }
      if (up) jbase += half;
      step<K + 1>(v, lane, jbase);
    }
  }
  // Sums v over the SPW stack lanes that share p.  Scatter form: lane keeps elements [jbase, jbase + R).
  __device__ static __forceinline__ void run(float (&v)[S::E], int lane, int& jbase) {
    jbase = 0;
    if constexpr (kScatter) {
      step<0>(v, lane, jbase);
    } else {
#pragma unroll
      for (int mask = S::P; mask < kWarp; mask <<= 1) {
#pragma unroll
        for (int j = 0; j < S::E; ++j) v[j] += __shfl_xor_sync(0xffffffffu, v[j], mask);
      }
    }
  }
};

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
  return v;
}

template <typename S>
__global__ void __launch_bounds__(kFwdThreads, (S::E >= 128 ? 3 : 4))
sorf_backward_kernel(const float* __restrict__ x, const int32_t* __restrict__ elem,
                     const int32_t* __restrict__ mol_off, int n_atoms, int n_mol, int n_s, int T, float c_rev,
                     float c, const uint32_t* __restrict__ sign_bits, const float* __restrict__ bias_rev,
                     const float* __restrict__ alpha_s, float* __restrict__ g_out,
                     double* __restrict__ energy_acc, int chunk, int n_chunks, int n_sg) {
  using SR = StackReduce<S>;
  extern __shared__ float4 xchg_smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  float4* xb = xchg_smem + warp * kXchgFloat4PerWarp;  // cross-lane scratch (P > 1 only)
  const long long task = (long long)blockIdx.x * (kFwdThreads / kWarp) + warp;
  if (task >= n_chunks) return;
  const int p = lane % S::P, sl = lane / S::P;
  const int n_gl = n_s * S::P;
  // fixed-size atom chunks (equal work per warp); molecule changes inside a chunk only flush the energy partial
  const int a_begin = (int)task * chunk;
  const int a_end = a_begin + chunk < n_atoms ? a_begin + chunk : n_atoms;
  if (a_begin >= a_end) return;

  int mol = owner_molecule(mol_off, n_mol, a_begin);
  int mol_hi = __ldg(mol_off + mol + 1);
  float epart = 0.f;
  const float4* bias4 = reinterpret_cast<const float4*>(bias_rev);
  const float4* alpha4 = reinterpret_cast<const float4*>(alpha_s);

#pragma unroll 1
  for (int a = a_begin; a < a_end; ++a) {
    if (a >= mol_hi) {
      if (energy_acc) {
        const float tot = warp_sum(epart);
        if (lane == 0) atomicAdd(energy_acc + mol, (double)tot);
      }
      epart = 0.f;
      do { ++mol; mol_hi = __ldg(mol_off + mol + 1); } while (a >= mol_hi);
    }
    const int e = __ldg(elem + a);
    float gacc[SR::R];
#pragma unroll
    for (int i = 0; i < SR::R; ++i) gacc[i] = 0.f;
    int jbase = 0;
#pragma unroll 1
    for (int sg = 0; sg < n_sg; ++sg) {
      const int s_raw = sg * S::SPW + sl;
      const bool valid = s_raw < n_s;
      const int gl = (valid ? s_raw : n_s - 1) * S::P + p;
      float v[S::E];
      load_row<S>(v, x + (size_t)a * S::d, p);
      const float4* b4 = bias4 + (size_t)e * S::E4 * n_gl + gl;
      const float4* al4 = alpha4 + gl;
      // Forward chain, sin/cos, transposed chain as ONE loop over 2T+1 phases so that the unrolled butterfly and
      // sign-flip code exist once (the straight-line version overflowed the instruction cache: 37 % no-instruction
      // stalls).  Phase i < T: S_i then H.  Phase T: u -> (energy, q) then H.  Phase T < i < 2T: S_{2T-i} then H.
      // Phase 2T: S_0 only.   [ (H S_{T-1} ... H S_0) x ;  S_0 H S_1 H ... S_{T-1} H q ]
#pragma unroll 1
      for (int i = 0; i <= 2 * T; ++i) {
        if (i == T) {
#pragma unroll
          for (int q = 0; q < S::E4; ++q) {
            const float4 b = __ldg(b4 + (size_t)q * n_gl);
            float4 al = __ldg(al4 + (size_t)q * n_gl);
            if (!valid) al = make_float4(0.f, 0.f, 0.f, 0.f);
            const float f0 = frac_rev(fmaf(v[4 * q + 0], c_rev, b.x));
            const float f1 = frac_rev(fmaf(v[4 * q + 1], c_rev, b.y));
            const float f2 = frac_rev(fmaf(v[4 * q + 2], c_rev, b.z));
            const float f3 = frac_rev(fmaf(v[4 * q + 3], c_rev, b.w));
            epart = fmaf(al.x, cos_rev(f0), epart); epart = fmaf(al.y, cos_rev(f1), epart);
            epart = fmaf(al.z, cos_rev(f2), epart); epart = fmaf(al.w, cos_rev(f3), epart);
            v[4 * q + 0] = -al.x * sin_rev(f0); v[4 * q + 1] = -al.y * sin_rev(f1);
            v[4 * q + 2] = -al.z * sin_rev(f2); v[4 * q + 3] = -al.w * sin_rev(f3);
          }
        } else {
          const int t = i < T ? i : 2 * T - i;
          uint32_t w[S::EW];
          load_sign_words<S>(w, sign_bits, e, t, T, n_gl, gl);
          apply_signs<S>(v, w);
        }
        if (i < 2 * T) fwht<S, true>(v, p, xb, lane);
      }
      SR::run(v, lane, jbase);
#pragma unroll
      for (int i = 0; i < SR::R; ++i) gacc[i] += v[i];
    }
    if (g_out && (SR::kScatter || sl == 0)) {
      float* dst = g_out + (size_t)a * S::d + p * S::E + jbase;
#pragma unroll
      for (int i = 0; i < SR::R; ++i) dst[i] = c * gacc[i];
    }
  }
  if (energy_acc) {
    const float tot = warp_sum(epart);
    if (lane == 0) atomicAdd(energy_acc + mol, (double)tot);
  }
}

// ------------------------------------------------------------------------------------------------
// Force rows (a7), dense gradient.  Warp task = (row r = 3*j + k, stack group).  The warp loops over the
// atoms I of the molecule that owns atom j: the gradient column dx_I[:, j, k] goes through the same chain as
// x (JVP of a linear map = the map itself), is weighted by the stored sqrt(2/D) sin(u_I + b) and summed over
// I in the shared-memory accumulators; the finished [SPW, d] slab of G row r is then written once.
//   G[r, l] = c * sum_I zs_I[l] * (H S_T ... H S_1 dx_I[:, j, k])[l]
// ------------------------------------------------------------------------------------------------
// `gt` is the gradient with each column made contiguous ([n, n, 3, d] = (I, j, k, m) per molecule, written by
// transpose_dense_kernel); the column of the next atom is staged in shared memory by a 1-D TMA bulk copy while
// the current one runs through the chain (2-deep ring per warp, one mbarrier per slot).
template <typename S>
struct ColStage {
  static constexpr int kSlice = S::E + 4;                 // floats per lane slice (+16 B: no bank conflicts for P > 1)
  static constexpr int kBufFloats = S::P * kSlice;        // one staged column
  static constexpr size_t kBytes = (size_t)(kFwdThreads / kWarp) * 2 * (kBufFloats * sizeof(float) + sizeof(uint64_t));
};

template <typename S>
__global__ void __launch_bounds__(kFwdThreads, (S::E >= 128 ? 3 : 4))
sorf_force_rows_dense_kernel(const int32_t* __restrict__ elem, const int32_t* __restrict__ mol_off, int n_atoms,
                             int n_mol, int n_s, int T, float c, const uint32_t* __restrict__ sign_bits,
                             const float* __restrict__ zs, const float* __restrict__ gt,
                             const int64_t* __restrict__ dense_off, float* __restrict__ G, int n_sg) {
  extern __shared__ float4 acc[];
  using CS = ColStage<S>;
  constexpr int kWarps = kFwdThreads / kWarp;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  float* colbuf = reinterpret_cast<float*>(acc + S::E4 * kFwdThreads) + warp * 2 * CS::kBufFloats;
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<float*>(acc + S::E4 * kFwdThreads) +
                                               kWarps * 2 * CS::kBufFloats) + warp * 2;
  float4* xb = reinterpret_cast<float4*>(reinterpret_cast<char*>(acc) + S::E * kFwdThreads * sizeof(float) +
                                         CS::kBytes) + warp * kXchgFloat4PerWarp;  // cross-lane scratch (P > 1)
  const long long task = (long long)blockIdx.x * kWarps + warp;
  if (task >= 3LL * n_atoms * n_sg) return;
  const int sg = (int)(task % n_sg);
  const long long r = task / n_sg;
  const int jg = (int)(r / 3), k = (int)(r % 3);
  const int p = lane % S::P, sl = lane / S::P;
  const int n_gl = n_s * S::P;
  const int s_raw = sg * S::SPW + sl;
  const int gl = (s_raw < n_s ? s_raw : n_s - 1) * S::P + p;

  const int M = owner_molecule(mol_off, n_mol, jg);
  const int a0 = __ldg(mol_off + M), n = __ldg(mol_off + M + 1) - a0;
  const int jl = jg - a0;
  // column (I, jl, k) of molecule M: d contiguous floats; consecutive I are 3*n*d floats apart
  const float* col0 = gt + __ldg(dense_off + M) + ((size_t)jl * 3 + k) * S::d;
  const size_t istride = (size_t)3 * n * S::d;

  if (lane == 0) {
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    fence_mbarrier_init();
  }
  __syncwarp();
  auto stage = [&](int I) {  // lane 0 only
    uint64_t* bar = &bars[I & 1];
    float* dst = colbuf + (I & 1) * CS::kBufFloats;
    mbar_expect_tx(bar, S::d * sizeof(float));
#pragma unroll
    for (int pp = 0; pp < S::P; ++pp)
      bulk_copy_g2s(dst + pp * CS::kSlice, col0 + (size_t)I * istride + pp * S::E, S::E * sizeof(float), bar);
  };
  if (lane == 0) stage(0);

  zero_acc<S>(acc, tid);
  const float4* zs4 = reinterpret_cast<const float4*>(zs);
#pragma unroll 1
  for (int I = 0; I < n; ++I) {
    if (lane == 0 && I + 1 < n) stage(I + 1);  // slot (I+1)&1 was last read in iteration I-1 (warp-synced below)
    const int e = __ldg(elem + a0 + I);
    mbar_wait(&bars[I & 1], (uint32_t)((I >> 1) & 1));
    float v[S::E];
    {
      const float4* src = reinterpret_cast<const float4*>(colbuf + (I & 1) * CS::kBufFloats + p * CS::kSlice);
#pragma unroll
      for (int q = 0; q < S::E4; ++q) {
        const float4 t = src[q];
        v[4 * q + 0] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
      }
    }
    __syncwarp();
    chain_forward<S>(v, sign_bits, e, T, n_gl, gl, p, xb, lane);
    const float4* z4 = zs4 + (size_t)(a0 + I) * S::E4 * n_gl + gl;
#pragma unroll
    for (int q = 0; q < S::E4; ++q) {
      const float4 z = __ldg(z4 + (size_t)q * n_gl);
      float4 ac = acc[q * kFwdThreads + tid];
      ac.x = fmaf(z.x, v[4 * q + 0], ac.x); ac.y = fmaf(z.y, v[4 * q + 1], ac.y);
      ac.z = fmaf(z.z, v[4 * q + 2], ac.z); ac.w = fmaf(z.w, v[4 * q + 3], ac.w);
      acc[q * kFwdThreads + tid] = ac;
    }
  }
  flush_slab<S>(acc, warp * kWarp, lane, G + (size_t)r * (size_t)n_s * S::d, sg, n_s, c, false);
}

// Force rows, neighbour-sparse gradient (A13): rows of different atoms collide, so contributions are added
// with atomics into a pre-zeroed G.  Warp task = (atom I, neighbour slot q, stack group), 3 columns each.
template <typename S>
__global__ void __launch_bounds__(kFwdThreads, (S::E >= 128 ? 3 : 4))
sorf_force_rows_neighbor_kernel(const int32_t* __restrict__ elem, int n_atoms, int n_s, int T, float c,
                                const uint32_t* __restrict__ sign_bits, const float* __restrict__ zs,
                                const int32_t* __restrict__ nbr_idx, const float* __restrict__ nbr_val, int K,
                                float* __restrict__ G, int n_sg) {
  extern __shared__ float4 xchg_smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  float4* xb = xchg_smem + warp * kXchgFloat4PerWarp;  // cross-lane scratch (P > 1 only)
  const long long task = (long long)blockIdx.x * (kFwdThreads / kWarp) + warp;
  if (task >= (long long)n_atoms * K * n_sg) return;
  const int sg = (int)(task % n_sg);
  const long long iq = task / n_sg;
  const int I = (int)(iq / K);
  const int jg = __ldg(nbr_idx + iq);
  if (jg < 0) return;
  const int p = lane % S::P, sl = lane / S::P;
  const int n_gl = n_s * S::P;
  const int s_raw = sg * S::SPW + sl;
  const bool valid = s_raw < n_s;
  const int gl = (valid ? s_raw : n_s - 1) * S::P + p;
  const int e = __ldg(elem + I);
  const float4* z4 = reinterpret_cast<const float4*>(zs) + (size_t)I * S::E4 * n_gl + gl;
  const float* val = nbr_val + (size_t)iq * S::d * 3;
#pragma unroll 1
  for (int k = 0; k < 3; ++k) {
    float v[S::E];
#pragma unroll
    for (int j = 0; j < S::E; ++j) v[j] = __ldg(val + (size_t)(p * S::E + j) * 3 + k);
    chain_forward<S>(v, sign_bits, e, T, n_gl, gl, p, xb, lane);
    if (valid) {
      float* dst = G + ((size_t)jg * 3 + k) * (size_t)n_s * S::d + (size_t)s_raw * S::d + p * S::E;
#pragma unroll
      for (int q = 0; q < S::E4; ++q) {
        const float4 z = __ldg(z4 + (size_t)q * n_gl);
        atomicAdd(dst + 4 * q + 0, c * z.x * v[4 * q + 0]); atomicAdd(dst + 4 * q + 1, c * z.y * v[4 * q + 1]);
        atomicAdd(dst + 4 * q + 2, c * z.z * v[4 * q + 2]); atomicAdd(dst + 4 * q + 3, c * z.w * v[4 * q + 3]);
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
  static constexpr size_t kXchgBytes = kWarpsPerBlock * Xchg<S>::kBytesPerWarp;

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
    const float c = c_of(p);
    const float c_rev = (float)((double)c / (2.0 * M_PI)), nrm = (float)sqrt(2.0 / (double)p->D);
    auto kern = zs_out ? sorf_forward_kernel<S, true> : sorf_forward_kernel<S, false>;
    QMLL_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kAccBytes));
    kern<<<grid, kFwdThreads, kAccBytes, st>>>(pr.x, pr.elem, pr.mol_off, n_atoms, pr.n_mol, n_s,
                                               p->n_transform, c_rev, nrm, t.sign_bits, t.bias_rev, Z, zs_out,
                                               chunk, n_chunks, n_sg);
    QMLL_LAUNCH_CHECK("sorf_forward_kernel");
    return QMLL_OK;
  }

  static int backward(const SorfProblem& pr, const SorfTables& t, float* g_out, double* energy_acc,
                      cudaStream_t st) {
    const qmll_sorf_params* p = pr.p;
    const int n_s = p->D / p->d, n_sg = (n_s + S::SPW - 1) / S::SPW;
    const int n_atoms = (int)pr.n_atoms;
    if (n_atoms == 0 || pr.n_mol == 0) return QMLL_OK;
    const int chunk = clampi((long long)n_atoms / (8LL * warp_slots()), 1, 8);
    const int n_chunks = (n_atoms + chunk - 1) / chunk;
    const unsigned grid = (unsigned)((n_chunks + kWarpsPerBlock - 1) / kWarpsPerBlock);
    const float c = c_of(p);
    const float c_rev = (float)((double)c / (2.0 * M_PI));
    sorf_backward_kernel<S><<<grid, kFwdThreads, kXchgBytes, st>>>(pr.x, pr.elem, pr.mol_off, n_atoms, pr.n_mol, n_s,
                                                          p->n_transform, c_rev, c, t.sign_bits, t.bias_rev,
                                                          t.alpha_s, g_out, energy_acc, chunk, n_chunks, n_sg);
    QMLL_LAUNCH_CHECK("sorf_backward_kernel");
    return QMLL_OK;
  }

  static int force_rows_dense(const SorfProblem& pr, const SorfTables& t, const float* zs, const float* dense,
                              const int64_t* dense_off, float* G, cudaStream_t st) {
    const qmll_sorf_params* p = pr.p;
    const int n_s = p->D / p->d, n_sg = (n_s + S::SPW - 1) / S::SPW;
    const int n_atoms = (int)pr.n_atoms;
    if (n_atoms == 0) return QMLL_OK;
    const long long tasks = 3LL * n_atoms * n_sg;
    const long long grid = (tasks + kWarpsPerBlock - 1) / kWarpsPerBlock;
    if (grid > 0x7fffffffLL) return QMLL_ERR_UNSUPPORTED;
    auto kern = sorf_force_rows_dense_kernel<S>;
    const size_t smem = kAccBytes + ColStage<S>::kBytes;
    QMLL_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<(unsigned)grid, kFwdThreads, smem, st>>>(pr.elem, pr.mol_off, n_atoms, pr.n_mol, n_s,
                                                         p->n_transform, c_of(p), t.sign_bits, zs, dense,
                                                         dense_off, G, n_sg);
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
  int sorf_backward_##TAG(const SorfProblem&, const SorfTables&, float*, double*, cudaStream_t);               \
  int sorf_force_rows_dense_##TAG(const SorfProblem&, const SorfTables&, const float*, const float*,           \
                                  const int64_t*, float*, cudaStream_t);                                       \
  int sorf_force_rows_neighbor_##TAG(const SorfProblem&, const SorfTables&, const float*, const int32_t*,      \
                                     const float*, int, float*, cudaStream_t);

#define QMLL_DEFINE_SORF_SHAPE_D(TAG, D_) QMLL_DEFINE_SORF_SHAPE(TAG, shape_E(D_), shape_P(D_))
#define QMLL_DEFINE_SORF_SHAPE(TAG, E_, P_)                                                                   \
  int sorf_forward_##TAG(const SorfProblem& pr, const SorfTables& t, float* Z, float* zs, cudaStream_t st) {   \
    return SorfLaunch<Shape<E_, P_>>::forward(pr, t, Z, zs, st);                                               \
  }                                                                                                            \
  int sorf_backward_##TAG(const SorfProblem& pr, const SorfTables& t, float* g, double* en, cudaStream_t st) { \
    return SorfLaunch<Shape<E_, P_>>::backward(pr, t, g, en, st);                                              \
  }                                                                                                            \
  int sorf_force_rows_dense_##TAG(const SorfProblem& pr, const SorfTables& t, const float* zs,                 \
                                  const float* dense, const int64_t* off, float* G, cudaStream_t st) {         \
    return SorfLaunch<Shape<E_, P_>>::force_rows_dense(pr, t, zs, dense, off, G, st);                          \
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
