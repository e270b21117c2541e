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
constexpr int kPredThreads = 256; // predict with forces: 8 warps, one block per SM (chain + stream want ~250 registers)
constexpr int kEnergyThreads = 384; // energies only: 12 warps (no transposed chain, no accumulators: 168 registers)

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
// stream of others, and g never leaves the SM.  The block's warps step through the stack groups
// without a barrier (measured: forcing them onto the same group with __syncthreads costs 5-8 %).
// energy_acc[mol] (double, pre-zeroed) receives one atomicAdd per atom.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
  return v;
}

constexpr int kGradGOut = 3;   // internal layout value: write g = dE/dx instead of contracting (qmll_sorf_backward_g)
struct GradView {          // qmll_grad flattened for the device
  int layout;              // QMLL_GRAD_NONE / DENSE / NEIGHBOR
  const float* dense;
  const int64_t* dense_off;
  const int32_t* nbr_idx;
  const float* nbr_val;
  int K;
};

// F[a0 + j, k] += sum_m gbuf[m] * dx[Il][m][3 j + k]   (dense layout, A12): lane = up to three columns (col, col + 32,
// col + 64), rows streamed 16 deep, i.e. up to 48 independent loads in flight per lane: the stream is latency-bound
// per warp, and the warp holds no chain state while it runs (its 128 vector registers are free).
template <typename S>
__device__ __forceinline__ void contract_dense_atom(const float* __restrict__ gbuf, const float* __restrict__ blk,
                                                    int ncol, float* __restrict__ Fmol, int lane) {
  for (int c0 = 0; c0 < ncol; c0 += 3 * kWarp) {
    const int col0 = c0 + lane, col1 = col0 + kWarp, col2 = col1 + kWarp;
    const bool ok0 = col0 < ncol, ok1 = col1 < ncol, ok2 = col2 < ncol;
    const float* p0 = blk + (ok0 ? col0 : 0);
    const float* p1 = blk + (ok1 ? col1 : 0);
    const float* p2 = blk + (ok2 ? col2 : 0);
    float s0 = 0.f, s1 = 0.f, s2 = 0.f;
#pragma unroll 1
    for (int m = 0; m < S::d; m += 16) {
      float a[16], b[16], c[16];
#pragma unroll
      for (int u = 0; u < 16; ++u) {
        a[u] = __ldcs(p0 + (size_t)(m + u) * ncol);
        b[u] = __ldcs(p1 + (size_t)(m + u) * ncol);
        c[u] = __ldcs(p2 + (size_t)(m + u) * ncol);
      }
#pragma unroll
      for (int u = 0; u < 16; u += 4) {
        const float4 g = *reinterpret_cast<const float4*>(gbuf + m + u);
        s0 = fmaf(g.x, a[u], s0); s1 = fmaf(g.x, b[u], s1); s2 = fmaf(g.x, c[u], s2);
        s0 = fmaf(g.y, a[u + 1], s0); s1 = fmaf(g.y, b[u + 1], s1); s2 = fmaf(g.y, c[u + 1], s2);
        s0 = fmaf(g.z, a[u + 2], s0); s1 = fmaf(g.z, b[u + 2], s1); s2 = fmaf(g.z, c[u + 2], s2);
        s0 = fmaf(g.w, a[u + 3], s0); s1 = fmaf(g.w, b[u + 3], s1); s2 = fmaf(g.w, c[u + 3], s2);
      }
    }
    if (ok0) atomicAdd(Fmol + col0, s0);
    if (ok1) atomicAdd(Fmol + col1, s1);
    if (ok2) atomicAdd(Fmol + col2, s2);
  }
}

// F[j, k] += sum_m gbuf[m] * val[q][m][k], j = nbr_idx[a, q]   (neighbour layout, A13; duplicates and self add,
// -1 = padding): each [d, 3] block is 3d contiguous floats; a lane takes 12 of them (4 values of m) per step, and
// kNbrBatch neighbour blocks are in flight at once (the stream is latency-bound per warp).
constexpr int kNbrBatch = 4;
template <typename S>
__device__ __forceinline__ void contract_neighbor_atom(const float* __restrict__ gbuf, const int32_t* __restrict__ idx,
                                                       const float* __restrict__ val, int K, float* __restrict__ F,
                                                       int lane) {
  constexpr int G = S::d / 4;                          // groups of 12 floats per block
  constexpr int GPL = (G + kWarp - 1) / kWarp;         // groups per lane
  constexpr int NB = GPL <= 2 ? kNbrBatch : (GPL <= 4 ? 2 : 1);
  const float4* g4 = reinterpret_cast<const float4*>(gbuf);
  float4 gv[GPL];
#pragma unroll
  for (int t = 0; t < GPL; ++t) {
    const int grp = lane + kWarp * t;
    gv[t] = (G % kWarp == 0 || grp < G) ? g4[grp] : make_float4(0.f, 0.f, 0.f, 0.f);
  }
#pragma unroll 1
  for (int q0 = 0; q0 < K; q0 += NB) {
    int j[NB];
    float4 f[NB][GPL][3];
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      j[b] = (q0 + b < K) ? __ldg(idx + q0 + b) : -1;
      const float4* v4 = reinterpret_cast<const float4*>(val + (size_t)(q0 + b) * S::d * 3);
#pragma unroll
      for (int t = 0; t < GPL; ++t) {
        const int grp = lane + kWarp * t;
        if (j[b] >= 0 && (G % kWarp == 0 || grp < G)) {
          f[b][t][0] = __ldcs(v4 + 3 * grp); f[b][t][1] = __ldcs(v4 + 3 * grp + 1); f[b][t][2] = __ldcs(v4 + 3 * grp + 2);
        } else {
          f[b][t][0] = f[b][t][1] = f[b][t][2] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
      }
    }
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      float ax = 0.f, ay = 0.f, az = 0.f;
#pragma unroll
      for (int t = 0; t < GPL; ++t) {
        const float4 g = gv[t], f0 = f[b][t][0], f1 = f[b][t][1], f2 = f[b][t][2];
        ax = fmaf(g.x, f0.x, ax); ay = fmaf(g.x, f0.y, ay); az = fmaf(g.x, f0.z, az);
        ax = fmaf(g.y, f0.w, ax); ay = fmaf(g.y, f1.x, ay); az = fmaf(g.y, f1.y, az);
        ax = fmaf(g.z, f1.z, ax); ay = fmaf(g.z, f1.w, ay); az = fmaf(g.z, f2.x, az);
        ax = fmaf(g.w, f2.y, ax); ay = fmaf(g.w, f2.z, ay); az = fmaf(g.w, f2.w, az);
      }
#pragma unroll
      for (int m = 16; m > 0; m >>= 1) {
        ax += __shfl_xor_sync(0xffffffffu, ax, m);
        ay += __shfl_xor_sync(0xffffffffu, ay, m);
        az += __shfl_xor_sync(0xffffffffu, az, m);
      }
      if (lane == 0 && j[b] >= 0) {
        atomicAdd(F + (size_t)j[b] * 3 + 0, ax);
        atomicAdd(F + (size_t)j[b] * 3 + 1, ay);
        atomicAdd(F + (size_t)j[b] * 3 + 2, az);
      }
    }
  }
}

// L2 prefetch of [ptr, ptr + floats): 4 KB pieces spread over the lanes (cp.async.bulk.prefetch.L2; pieces stay
// inside the range, 16-byte aligned).
__device__ __forceinline__ void l2_prefetch_range(const float* ptr, size_t floats, int lane) {
  const uintptr_t b = ((uintptr_t)ptr + 15) & ~(uintptr_t)15, e = (uintptr_t)(ptr + floats) & ~(uintptr_t)15;
  for (uintptr_t q = b + (uintptr_t)lane * 4096; q < e; q += (uintptr_t)kWarp * 4096) {
    const uint32_t sz = e - q < 4096 ? (uint32_t)(e - q) : 4096u;
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(q), "r"(sz) : "memory");
  }
}

template <typename S>
struct PredSmem {
  static constexpr int kWarps = kPredThreads / kWarp;
  static constexpr size_t kAccBytes = (size_t)S::E * kWarp * sizeof(float);       // per warp: [E4][32] float4
  static constexpr size_t kBytes = kWarps * (kAccBytes + S::d * sizeof(float));   // + gbuf[d] per warp
};

template <typename S, bool kNeedG, int kThreads>
__global__ void __launch_bounds__(kThreads, 1)
sorf_predict_kernel(const float* __restrict__ x, const int32_t* __restrict__ elem,
                    const int32_t* __restrict__ mol_off, int n_atoms, int n_mol, int n_s, int T, float c,
                    const uint32_t* __restrict__ sign_bits, const float* __restrict__ bias_t,
                    const float* __restrict__ alpha_s, GradView grad, float* __restrict__ forces,
                    double* __restrict__ energy_acc, int atoms_per_block, int n_sg) {
  extern __shared__ float4 smem4[];
  constexpr int kWarps = kThreads / kWarp;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  float4* acc = smem4 + warp * (S::E4 * kWarp);                                           // [E4][32]
  float* gbuf = reinterpret_cast<float*>(smem4 + kWarps * (S::E4 * kWarp)) + warp * S::d;  // [d]
  const int p = lane % S::P;
  const int a_block = blockIdx.x * atoms_per_block;
  const int a_stop = a_block + atoms_per_block < n_atoms ? a_block + atoms_per_block : n_atoms;
  const float4* bias4 = reinterpret_cast<const float4*>(bias_t);
  const float4* alpha4 = reinterpret_cast<const float4*>(alpha_s);
  const f32x2 c2 = pk(c, c);

  int M = 0;
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
    // the molecule that owns the atom, found before the chain: a binary search for the warp's first atom, then a walk
    // (the warp's atoms increase; empty molecules are stepped over)
    if (have && (energy_acc != nullptr || (kNeedG && grad.layout == QMLL_GRAD_DENSE))) {
      if (a0 == a_block) M = owner_molecule(mol_off, n_mol, a);
      else while (__ldg(mol_off + M + 1) <= a) ++M;
    }
#pragma unroll 1
    for (int sg = 0; sg < n_sg; ++sg) {
      if (!have) continue;
      if (kNeedG && sg == n_sg - 1) {
        // The atom's gradient block is streamed exactly once, after the chain, by this warp: ask for it in L2 when
        // the last stack group starts (early enough to land, late enough that the blocks of all resident warps --
        // 83 KB each on config 4 -- do not crowd L2).  Measured: config 4 inference 3.70 -> 3.58 ms, config 5 2.06 -> 1.94.
        if (grad.layout == QMLL_GRAD_DENSE) {
          const int lo = __ldg(mol_off + M), np_ = __ldg(mol_off + M + 1) - lo;
          l2_prefetch_range(grad.dense + __ldg(grad.dense_off + M) + (size_t)(a - lo) * S::d * 3 * np_,
                            (size_t)S::d * 3 * np_, lane);
        } else if (grad.layout == QMLL_GRAD_NEIGHBOR) {
          l2_prefetch_range(grad.nbr_val + (size_t)a * grad.K * S::d * 3, (size_t)grad.K * S::d * 3, lane);
        }
      }
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
        sign_fwht<S>(v, w, p);
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
    int m_lo = 0, n = 0;
    if (energy_acc != nullptr || (kNeedG && grad.layout == QMLL_GRAD_DENSE)) {
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
      } else if (grad.layout == QMLL_GRAD_NEIGHBOR) {
        contract_neighbor_atom<S>(gbuf, grad.nbr_idx + (size_t)a * grad.K,
                                  grad.nbr_val + (size_t)a * grad.K * S::d * 3, grad.K, forces, lane);
      } else {   // kGradGOut: no contraction, `forces` is g [n_atoms, d] = dE/dx (gbuf holds -dE/dx)
        for (int m = lane; m < S::d; m += kWarp) forces[(size_t)a * S::d + m] = -gbuf[m];
      }
      __syncwarp();
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Force rows (a7), dense gradient.  Warp task = (row r = 3*j + k, stack group); the four warps of a block take
// four consecutive rows of the same stack group.  The warp loops over the atoms I of the molecule that owns
// atom j: the gradient column dx_I[:, j, k] goes through the same chain as x (JVP of a linear map = the map
// itself), is weighted by sqrt(2/D) sin(u_I + b) of that (atom, stack group) and summed over I in the warp's
// shared-memory accumulators; the finished [SPW, d] slab of G row r is then written once.
//   G[r, l] = c * sum_I zs_I[l] * (H S_T ... H S_1 dx_I[:, j, k])[l]
// `gt` is the gradient with each column made contiguous ([n, n, 3, d] = (I, j, k, m) per molecule, written by
// transpose_dense_kernel); the column of the next atom is staged in shared memory by a 1-D TMA bulk copy while
// the current one runs through the chain (2-slot ring per warp, one mbarrier per slot).  The sin table of
// (I, stack group) -- E*128 bytes, written by the forward kernel -- is read through L1: every warp prefetches the
// table of the NEXT atom into L1 before it starts the chain of the current one, and the warps of a block (same
// molecule, same stack group) find each other's lines there.  The warps are independent (no block-level barrier):
// measured, coupling them through a shared staged table put their shared-memory phases in lockstep and cost 15 %.
// ------------------------------------------------------------------------------------------------
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
  // block -> (group of kWarps consecutive rows, stack group); warp -> row
  const int sg = blockIdx.x % n_sg;
  const long long r = (long long)(blockIdx.x / n_sg) * kWarps + warp;
  if (r >= 3LL * n_atoms) return;
  const int jg = (int)(r / 3);
  const int p = lane % S::P;

  const int M = owner_molecule(mol_off, n_mol, jg);
  const int a0 = __ldg(mol_off + M), n = __ldg(mol_off + M + 1) - a0;
  const int rl = (int)(r - 3LL * a0);             // local row 3*jl + k of molecule M
  // column (I, jl, k) of molecule M: d contiguous floats of gt; consecutive I are 3*n*d floats apart
  const float* col0 = gt + __ldg(dense_off + M) + (size_t)rl * S::d;
  const size_t istride = (size_t)3 * n * S::d;
  const float4* zs4 = reinterpret_cast<const float4*>(zs) + ((size_t)a0 * n_sg + sg) * (S::E4 * kWarp) + lane;
  const size_t zs_stride = (size_t)n_sg * (S::E4 * kWarp);   // float4 per atom

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
  auto prefetch_zs = [&](int I) {  // the (atom, stack group) table is E*128 contiguous bytes = E lines of 128 B
    const char* base = reinterpret_cast<const char*>(zs4 - lane + (size_t)I * zs_stride);
#pragma unroll
    for (int k = 0; k < S::E / kWarp; ++k)
      asm volatile("prefetch.global.L1 [%0];" ::"l"(base + (size_t)(k * kWarp + lane) * 128));
  };
  if (lane == 0) stage(0);
  prefetch_zs(0);

  zero_acc<S, kFwdThreads>(acc, tid);
#pragma unroll 1
  for (int I = 0; I < n; ++I) {
    if (I + 1 < n) {
      if (lane == 0) stage(I + 1);  // slot (I+1)&1 was last read in iteration I-1 (warp-synced below)
      prefetch_zs(I + 1);
    }
    const int e = __ldg(elem + a0 + I);
    mbar_wait(&bars[I & 1], (uint32_t)((I >> 1) & 1));
    f32x2 v[S::E2];
    load_row<S>(v, colbuf + (I & 1) * CS::kBufFloats + p * 4, p);   // slices are kSlice = E + 4 floats apart
    __syncwarp();
    chain_forward<S>(v, sign_bits, e, T, n_sg, sg, lane);
    const float4* z4 = zs4 + (size_t)I * zs_stride;
#pragma unroll
    for (int q = 0; q < S::E4; ++q) {
      const float4 z = __ldg(z4 + q * kWarp);
      float4 ac = acc[q * kFwdThreads + tid];
      f32x2 a01 = fma2(pk(z.x, z.y), v[2 * q], pk(ac.x, ac.y));
      f32x2 a23 = fma2(pk(z.z, z.w), v[2 * q + 1], pk(ac.z, ac.w));
      upk(a01, ac.x, ac.y);
      upk(a23, ac.z, ac.w);
      acc[q * kFwdThreads + tid] = ac;
    }
  }
  flush_slab<S, kFwdThreads>(acc, warp * kWarp, lane, G + (size_t)r * (size_t)n_s * S::d, sg, n_s, c, false);
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
    const int threads = forces ? kPredThreads : kEnergyThreads, n_warps = threads / kWarp;
    const int n_sm = device_sm_count();
    int apb = (n_atoms + n_sm - 1) / n_sm;
    apb = (apb + n_warps - 1) / n_warps * n_warps;
    const unsigned grid = (unsigned)((n_atoms + apb - 1) / apb);
    auto kern = forces ? sorf_predict_kernel<S, true, kPredThreads> : sorf_predict_kernel<S, false, kEnergyThreads>;
    const size_t smem = forces ? PredSmem<S>::kBytes : 0;
    QMLL_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<grid, threads, smem, st>>>(pr.x, pr.elem, pr.mol_off, n_atoms, pr.n_mol, n_s, p->n_transform,
                                           c_of(p), t.sign_bits, t.bias_t, t.alpha_s, gv, forces, energy_acc, apb,
                                           n_sg);
    QMLL_LAUNCH_CHECK("sorf_predict_kernel");
    return QMLL_OK;
  }

  static int force_rows_dense(const SorfProblem& pr, const SorfTables& t, const float* zs, const float* dense_t,
                              const int64_t* dense_off, float* G, cudaStream_t st) {
    const qmll_sorf_params* p = pr.p;
    const int n_s = p->D / p->d, n_sg = (n_s + S::SPW - 1) / S::SPW;
    const long long n_atoms = pr.n_atoms;
    if (n_atoms == 0) return QMLL_OK;
    const long long grid = (3 * n_atoms + kWarpsPerBlock - 1) / kWarpsPerBlock * n_sg;
    if (grid > 0x7fffffffLL) return QMLL_ERR_UNSUPPORTED;
    auto kern = sorf_force_rows_dense_kernel<S>;
    const size_t smem = kAccBytes + ColStage<S>::kBytes;
    QMLL_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<(unsigned)grid, kFwdThreads, smem, st>>>(pr.elem, pr.mol_off, (int)n_atoms, pr.n_mol, n_s, p->n_transform,
                                                    c_of(p), t.sign_bits, zs, dense_t, dense_off, G, n_sg);
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
                                  const int64_t*, float*, cudaStream_t);                                       \
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
