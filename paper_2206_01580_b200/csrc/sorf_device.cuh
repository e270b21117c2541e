// sorf_device.cuh -- register-resident Walsh-Hadamard / sign chain of the SORF map (eq. 20, PAPER.md
// L158-167) and the thread <-> data mapping shared by the forward, backward and force-row kernels.
//
// Mapping.  One descriptor vector of length d = E*P lives in P adjacent lanes of a warp, E elements
// per lane in registers (E <= 128): element m = p*E + j, p = lane % P, j = register index.  A warp
// therefore carries SPW = 32/P independent vectors, one per SORF stack s ("stack lane" sl = lane / P):
// all of them are transforms of the SAME input row x_I with different sign diagonals, so x_I is a
// broadcast load and no inter-lane traffic is needed for the log2(E) low butterfly stages.  The
// log2(P) high stages (d > 128 only) exchange through a small shared-memory scratch (see fwht).  For d <= 128 the whole
// H*D3*H*D2*H*D1 chain of a stack is register-local.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace qmll {

constexpr int kWarp = 32;

// Elements per lane: the whole vector for d <= QMLL_MAX_E, else QMLL_MAX_E with P = d / QMLL_MAX_E lanes per vector.
#ifndef QMLL_MAX_E
#define QMLL_MAX_E 128
#endif
constexpr int shape_E(int d) { return d < QMLL_MAX_E ? d : QMLL_MAX_E; }
constexpr int shape_P(int d) { return d / shape_E(d); }
constexpr int ilog2(int v) { return v <= 1 ? 0 : 1 + ilog2(v >> 1); }

template <int E_, int P_>
struct Shape {
  static constexpr int E = E_;             // elements per lane
  static constexpr int P = P_;             // lanes per vector
  static constexpr int d = E_ * P_;        // descriptor length
  static constexpr int SPW = kWarp / P_;   // stacks per warp
  static constexpr int EW = (E_ + 31) / 32;  // 32-bit sign words per lane and transform
  static constexpr int E4 = E_ / 4;        // float4 groups per lane
  static_assert(E_ >= 16 && E_ <= 128 && (E_ & (E_ - 1)) == 0, "E");
  static_assert(P_ >= 1 && P_ <= 16 && (P_ & (P_ - 1)) == 0, "P");
};

// Per-warp shared-memory scratch for the cross-lane butterfly stages (P > 1): 32 elements per lane at a time.
constexpr int kXchgFloat4PerWarp = 8 * kWarp;  // 4 KB
template <typename S>
struct Xchg {
  static constexpr size_t kBytesPerWarp = S::P > 1 ? kXchgFloat4PerWarp * sizeof(float4) : 0;
};

// v <- H_d v (unnormalised, natural order): any order of the butterfly stages gives the same matrix.
// The log2(E) low stages are register-local.  The log2(P) high stages pair lane p with lane p ^ h: the partner's
// values come through the warp's shared-memory scratch as float4 (8 LDS.128 deliver 32 operands, which keeps the
// FFMAs fed; one SHFL per element left them waiting on the shuffle latency -- 29 % short-scoreboard stalls).
// kSmem selects the exchange path: the backward kernel (no other shared memory) uses it; the forward and force-row
// kernels keep one SHFL + FFMA per element, because 16 KB more shared memory per block would cost them a resident
// block per SM (their accumulators already take 64 KB).
template <typename S, bool kSmem>
__device__ __forceinline__ void fwht(float (&v)[S::E], int p, float4* xb, int lane) {
#pragma unroll
  for (int h = 1; h < S::E; h <<= 1) {
#pragma unroll
    for (int i = 0; i < S::E; i += 2 * h) {
#pragma unroll
      for (int j = i; j < i + h; ++j) {
        float a = v[j], b = v[j + h];
        v[j] = a + b;
        v[j + h] = a - b;
      }
    }
  }
  if constexpr (S::P > 1) {
#pragma unroll
    for (int h = 1; h < S::P; h <<= 1) {
      const float sg = (p & h) ? -1.0f : 1.0f;  // upper partner holds (lower - upper)
      if constexpr (!kSmem) {
#pragma unroll
        for (int j = 0; j < S::E; ++j) {
          float o = __shfl_xor_sync(0xffffffffu, v[j], h);
          v[j] = fmaf(v[j], sg, o);
        }
        continue;
      }
      constexpr int kChunk = S::E < 32 ? S::E : 32;
#pragma unroll
      for (int c = 0; c < S::E; c += kChunk) {
#pragma unroll
        for (int q = 0; q < kChunk / 4; ++q)
          xb[q * kWarp + lane] = make_float4(v[c + 4 * q], v[c + 4 * q + 1], v[c + 4 * q + 2], v[c + 4 * q + 3]);
        __syncwarp();
#pragma unroll
        for (int q = 0; q < kChunk / 4; ++q) {
          const float4 o = xb[q * kWarp + (lane ^ h)];
          v[c + 4 * q + 0] = fmaf(v[c + 4 * q + 0], sg, o.x);
          v[c + 4 * q + 1] = fmaf(v[c + 4 * q + 1], sg, o.y);
          v[c + 4 * q + 2] = fmaf(v[c + 4 * q + 2], sg, o.z);
          v[c + 4 * q + 3] = fmaf(v[c + 4 * q + 3], sg, o.w);
        }
        __syncwarp();
      }
    }
  }
}

// v <- S .* v with the E sign bits of this lane packed in w[] (bit set = -1): one shift + one LOP3.
template <typename S>
__device__ __forceinline__ void apply_signs(float (&v)[S::E], const uint32_t (&w)[S::EW]) {
#pragma unroll
  for (int j = 0; j < S::E; ++j) {
    uint32_t m = (w[j >> 5] << (31 - (j & 31))) & 0x80000000u;
    v[j] = __uint_as_float(__float_as_uint(v[j]) ^ m);
  }
}

template <typename S>
__device__ __forceinline__ void load_sign_words(uint32_t (&w)[S::EW], const uint32_t* __restrict__ sign_bits,
                                                int e, int t, int T, int n_gl, int gl) {
#pragma unroll
  for (int k = 0; k < S::EW; ++k) w[k] = __ldg(sign_bits + ((size_t)(e * T + t) * S::EW + k) * n_gl + gl);
}

// v <- x_I[p*E .. p*E+E): the same address in all lanes that share p (broadcast).
template <typename S>
__device__ __forceinline__ void load_row(float (&v)[S::E], const float* __restrict__ row, int p) {
  const float4* src = reinterpret_cast<const float4*>(row + p * S::E);
#pragma unroll
  for (int q = 0; q < S::E4; ++q) {
    float4 t = __ldg(src + q);
    v[4 * q + 0] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
  }
}

// One stack of eq. 20 without the constant c:  v <- H S_{T-1} ... H S_0 v   (sign flip, then H: L268, A4)
template <typename S>
__device__ __forceinline__ void chain_forward(float (&v)[S::E], const uint32_t* __restrict__ sign_bits, int e,
                                              int T, int n_gl, int gl, int p, float4* xb, int lane) {
  for (int t = 0; t < T; ++t) {
    uint32_t w[S::EW];
    load_sign_words<S>(w, sign_bits, e, t, T, n_gl, gl);
    apply_signs<S>(v, w);
    fwht<S, false>(v, p, xb, lane);
  }
}

// Transposed stack: v <- S_0 H ... S_{T-1} H v   (H symmetric).
template <typename S>
__device__ __forceinline__ void chain_transposed(float (&v)[S::E], const uint32_t* __restrict__ sign_bits,
                                                 int e, int T, int n_gl, int gl, int p, float4* xb, int lane) {
  for (int t = T - 1; t >= 0; --t) {
    uint32_t w[S::EW];
    load_sign_words<S>(w, sign_bits, e, t, T, n_gl, gl);
    fwht<S, false>(v, p, xb, lane);
    apply_signs<S>(v, w);
  }
}

// Fractional part in revolutions, |f| <= 0.5, for |t| < 2^22 (arguments here are a few revolutions).
__device__ __forceinline__ float frac_rev(float t) {
  float r = (t + 12582912.0f) - 12582912.0f;  // round to nearest integer (exact)
  return t - r;
}
// cos / sin of 2*pi*f for |f| <= 0.5 on the MUFU unit (abs. error ~4e-7 on this range).
__device__ __forceinline__ float cos_rev(float f) { return __cosf(f * 6.283185307179586f); }
__device__ __forceinline__ float sin_rev(float f) { return __sinf(f * 6.283185307179586f); }

// Smallest M with mol_off[M+1] > a, i.e. the molecule that owns atom a (skips empty molecules).
__device__ __forceinline__ int owner_molecule(const int32_t* __restrict__ mol_off, int n_mol, int a) {
  int lo = 0, hi = n_mol - 1;
  while (lo < hi) {
    int mid = (lo + hi) >> 1;
    if (__ldg(mol_off + mid + 1) > a) hi = mid; else lo = mid + 1;
  }
  return lo;
}
// First molecule start >= a (or n_atoms if none).
__device__ __forceinline__ int next_molecule_start(const int32_t* __restrict__ mol_off, int n_mol, int a) {
  int lo = 0, hi = n_mol;  // smallest M in [0, n_mol] with mol_off[M] >= a
  while (lo < hi) {
    int mid = (lo + hi) >> 1;
    if (__ldg(mol_off + mid) >= a) hi = mid; else lo = mid + 1;
  }
  return __ldg(mol_off + lo);
}
// Task c covers atoms [cut(c), cut(c+1)): cuts snap forward to a molecule start when one lies inside the
// chunk, so molecules no longer than a chunk are never split; long molecules are cut at chunk multiples.
__device__ __forceinline__ int chunk_cut(const int32_t* __restrict__ mol_off, int n_mol, int n_atoms, int c,
                                         int chunk) {
  long long a = (long long)c * chunk;
  if (a >= n_atoms) return n_atoms;
  int cand = next_molecule_start(mol_off, n_mol, (int)a);
  return (cand < a + chunk) ? cand : (int)a;
}

}  // namespace qmll
