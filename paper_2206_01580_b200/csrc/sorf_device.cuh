// sorf_device.cuh -- register-resident Walsh-Hadamard / sign chain of the SORF map (eq. 20, PAPER.md
// L158-167) and the thread <-> data mapping shared by the forward, predict and force-row kernels.
//
// Mapping.  One descriptor vector of length d = E*P lives in P adjacent lanes of a warp, E elements
// per lane in registers (E <= 128): element m = p*E + j, p = lane % P, j = register index.  A warp
// therefore carries SPW = 32/P independent vectors, one per SORF stack s ("stack lane" sl = lane / P):
// all of them are transforms of the SAME input row x_I with different sign diagonals, so x_I is a
// broadcast load and no inter-lane traffic is needed for the log2(E) low butterfly stages.  The
// log2(P) high stages (d > 128 only) are one SHFL pair + one packed FMA per element pair.
//
// Arithmetic.  The kernels are bound by fp32 add issue (measured on B200, profiles/peaks_r2.json: 128 FADD per
// clock and SM, one instruction issued per clock and scheduler).  The elements of a lane are therefore kept as
// PAIRS in 64-bit registers and the butterflies use the packed add.f32x2 / sub.f32x2 (FADD2: two adds per issue
// slot at the same adds-per-clock), which frees issue slots for the sign flips (integer pipe), the loads and the
// MUFU work: the chain runs at ~91 % of the FADD peak instead of ~78 % (7 FADD + 2 integer ops per element).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace qmll {

constexpr int kWarp = 32;

// Elements per lane: the whole vector for d <= 128, else 128 with P = d / 128 lanes per vector.
constexpr int kMaxE = 128;
constexpr int shape_E(int d) { return d < kMaxE ? d : kMaxE; }
constexpr int shape_P(int d) { return d / shape_E(d); }
constexpr int ilog2(int v) { return v <= 1 ? 0 : 1 + ilog2(v >> 1); }

template <int E_, int P_>
struct Shape {
  static constexpr int E = E_;             // elements per lane
  static constexpr int P = P_;             // lanes per vector
  static constexpr int d = E_ * P_;        // descriptor length
  static constexpr int SPW = kWarp / P_;   // stacks per warp
  static constexpr int EW = (E_ + 31) / 32;  // 32-bit sign words per lane and transform
  static constexpr int E2 = E_ / 2;        // packed pairs per lane
  static constexpr int E4 = E_ / 4;        // float4 groups per lane
  static_assert(E_ >= 16 && E_ <= 128 && (E_ & (E_ - 1)) == 0, "E");
  static_assert(P_ >= 1 && P_ <= 16 && (P_ & (P_ - 1)) == 0, "P");
};

// ---- packed fp32 pairs (sm_100: FADD2 / FFMA2 / FMUL2) ---------------------------------------------
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk(float lo, float hi) {
  f32x2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void upk(f32x2 v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
  f32x2 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
__device__ __forceinline__ f32x2 shfl_xor2(f32x2 v, int mask) {
  float a, b;
  upk(v, a, b);
  return pk(__shfl_xor_sync(0xffffffffu, a, mask), __shfl_xor_sync(0xffffffffu, b, mask));
}

// v <- H_d (S .* v)  for one transform: S = the lane's E sign bits packed in w[] (bit set = -1), H unnormalised,
// natural order (any order of the butterfly stages gives the same matrix).  The sign flip (one shift + one LOP3 per
// element, integer pipe) is fused with the only butterfly stage that pairs the two halves of a register pair; the
// other log2(E) - 1 local stages are packed adds; the log2(P) cross-lane stages pair lane p with lane p ^ h.
// The local stages are emitted depth-first (transform the two halves of a block, then combine them), so that the
// integer sign work of later leaves sits next to the packed adds of earlier blocks in the instruction stream:
// one warp then keeps the integer pipe and the fp32 pipe busy at the same time instead of in alternating phases.
template <typename S, int LO, int N>
__device__ __forceinline__ void sign_fwht_block(f32x2 (&v)[S::E2], const uint32_t (&w)[S::EW]) {
  if constexpr (N == 1) {
    float a, b;
    upk(v[LO], a, b);
    constexpr int j = 2 * LO;
    a = __uint_as_float(__float_as_uint(a) ^ ((w[j >> 5] << (31 - (j & 31))) & 0x80000000u));
    b = __uint_as_float(__float_as_uint(b) ^ ((w[j >> 5] << (30 - (j & 31))) & 0x80000000u));
    v[LO] = pk(a + b, a - b);
  } else {
    sign_fwht_block<S, LO, N / 2>(v, w);
    sign_fwht_block<S, LO + N / 2, N / 2>(v, w);
#pragma unroll
    for (int j = LO; j < LO + N / 2; ++j) {
      if constexpr (N == S::E2) {
        // last local stage, in place: a <- a + b, b <- a - 2b (= old a - old b up to one rounding of a + b): the
        // values of the transform end in the registers they started in, so the loop over the transforms closes
        // without a register-to-register move per element (13 % of all issued instructions otherwise)
        v[j] = add2(v[j], v[j + N / 2]);
        v[j + N / 2] = fma2(v[j + N / 2], pk(-2.f, -2.f), v[j]);
      } else {
        const f32x2 a = v[j], b = v[j + N / 2];
        v[j] = add2(a, b);
        v[j + N / 2] = sub2(a, b);
      }
    }
  }
}

template <typename S>
__device__ __forceinline__ void sign_fwht(f32x2 (&v)[S::E2], const uint32_t (&w)[S::EW], int p) {
  sign_fwht_block<S, 0, S::E2>(v, w);
  if constexpr (S::P > 1) {
#pragma unroll
    for (int h = 1; h < S::P; h <<= 1) {
      const float sg = (p & h) ? -1.0f : 1.0f;  // upper partner holds (lower - upper)
      const f32x2 sg2 = pk(sg, sg);
#pragma unroll
      for (int i = 0; i < S::E2; ++i) v[i] = fma2(v[i], sg2, shfl_xor2(v[i], h));
    }
  }
}

// Model tables are stored per (element, stack group) in lane order, so that everything one warp needs for one
// stack group is contiguous and every access has a compile-time offset from one base pointer:
//   sign_bits[(((e*T + t)*n_sg + sg)*EW + k)*32 + lane]     bit i  <->  S[e, s, t, p*E + 32k + i] == -1
//   bias_t   [(((e*n_sg + sg)*E4 + q)*32 + lane)*4 + i]      =   b[e, s*d + p*E + 4q + i]
//   alpha_s  [((sg*E4 + q)*32 + lane)*4 + i]                 =   alpha[s*d + p*E + 4q + i] * sqrt(2/D)
// with s = sg*SPW + lane/P, p = lane%P; lanes whose stack s >= n_s (last group) hold zeros, so they contribute nothing.
template <typename S>
__device__ __forceinline__ void load_sign_words(uint32_t (&w)[S::EW], const uint32_t* __restrict__ sign_bits,
                                                int e, int t, int T, int n_sg, int sg, int lane) {
  const uint32_t* src = sign_bits + (((size_t)(e * T + t) * n_sg + sg) * S::EW) * kWarp + lane;
#pragma unroll
  for (int k = 0; k < S::EW; ++k) w[k] = __ldg(src + k * kWarp);
}

// v <- row[p*E .. p*E+E): the same address in all lanes that share p (broadcast); `row` may be global or shared.
template <typename S>
__device__ __forceinline__ void load_row(f32x2 (&v)[S::E2], const float* __restrict__ row, int p) {
  const f32x2* src = reinterpret_cast<const f32x2*>(row + p * S::E);   // 64-bit loads: one register pair each
#pragma unroll
  for (int q = 0; q < S::E2; ++q) v[q] = src[q];
}

// One stack of eq. 20 without the constant c:  v <- H S_{T-1} ... H S_0 v   (sign flip, then H: L268, A4)
template <typename S>
__device__ __forceinline__ void chain_forward(f32x2 (&v)[S::E2], const uint32_t* __restrict__ sign_bits, int e,
                                              int T, int n_sg, int sg, int lane) {
  const int p = lane % S::P;
#pragma unroll 1
  for (int t = 0; t < T; ++t) {
    uint32_t w[S::EW];
    load_sign_words<S>(w, sign_bits, e, t, T, n_sg, sg, lane);
    sign_fwht<S>(v, w, p);
  }
}

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
