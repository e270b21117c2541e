// project_kernels.cu -- NEXT row f2 of SURVEY.md section 8(f): the per-element PCA projection in front of the SORF map,
//   x_I[m] = sum_k rho_I[k] U[e_I, k, m]                       (rho_I^T U_e^{N_PCA}, eq. 21-22)
// and the same projection of a dense descriptor gradient (U is constant: d x_I / d r = (d rho_I / d r)^T U_e),
//   dx_I[m, j, c] = sum_k drho_I[k, j, c] U[e_I, k, m].
// Both are small grouped GEMMs [d x rep] x [rep x C] per atom (C = 1 resp. 3n) in plain fp32 FMAs: the work is
// n_atoms * rep * d * C MACs (config 4: 1.1e11 for the gradient, a few ms; 5e9 for x), the accuracy is that of an fp32
// dot product of length rep (~1e-6 relative), and the result feeds qmll_sorf_forward / qmll_predict unchanged.
// Mapping: lane = column (an atom for x, a (j, c) column for the gradient), warp = a range of outputs m; the lane
// keeps 32 accumulators in registers, its input value comes from a shared-memory tile, the U values of a k are the
// same for the whole warp (broadcast float4 loads through L1).
#include "qmll_common.cuh"
#include "sorf_device.cuh"

namespace qmll {

constexpr int kProjThreads = 256;   // 8 warps
constexpr int kProjK = 64;          // k-chunk staged in shared memory
constexpr int kProjM = 32;          // outputs per warp pass (register accumulators)

// acc[mm] += U[k][m0 + mm] * a  for k in the staged chunk; tile[k][lane] holds the lane's input values
__device__ __forceinline__ void proj_accumulate(float (&acc)[kProjM], const float (*tile)[33], int kc, int lane,
                                                const float* __restrict__ Uk /* U_e + k0*d + m0 */, int d) {
#pragma unroll 4
  for (int k = 0; k < kc; ++k) {
    const float a = tile[k][lane];
    const float4* u4 = reinterpret_cast<const float4*>(Uk + (size_t)k * d);
#pragma unroll
    for (int q = 0; q < kProjM / 4; ++q) {
      const float4 u = __ldg(u4 + q);
      acc[4 * q + 0] = fmaf(u.x, a, acc[4 * q + 0]); acc[4 * q + 1] = fmaf(u.y, a, acc[4 * q + 1]);
      acc[4 * q + 2] = fmaf(u.z, a, acc[4 * q + 2]); acc[4 * q + 3] = fmaf(u.w, a, acc[4 * q + 3]);
    }
  }
}

// x: block = 32 consecutive atoms (lane = atom).  Atoms of different elements use different matrices: the block
// runs once per element present in its tile, lanes of other elements are masked out.
__global__ void __launch_bounds__(kProjThreads)
project_x_kernel(const float* __restrict__ rho, const int32_t* __restrict__ elem, long long n_atoms, int rep, int d,
                 int n_elem, const float* __restrict__ U, float* __restrict__ x) {
  __shared__ float tile[kProjK][33];
  __shared__ int present[64];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long a = (long long)blockIdx.x * 32 + lane;
  const int e_lane = a < n_atoms ? __ldg(elem + a) : -1;
  for (int i = threadIdx.x; i < 64; i += kProjThreads) present[i] = 0;
  __syncthreads();
  if (warp == 0 && e_lane >= 0) present[e_lane & 63] = 1;   // n_elem <= 64 handled exactly; beyond that all are tried
  __syncthreads();
  for (int e = 0; e < n_elem; ++e) {
    if (n_elem <= 64 && !present[e]) continue;
    const float* Ue = U + (size_t)e * rep * d;
    // every warp makes the same number of passes (it helps staging the tile even if it owns no outputs in a pass)
    for (int mp = 0; mp < d; mp += (kProjThreads / 32) * kProjM) {
      const int m0 = mp + warp * kProjM;
      const int mw = m0 >= d ? 0 : (d - m0 < kProjM ? d - m0 : kProjM);
      float acc[kProjM];
#pragma unroll
      for (int i = 0; i < kProjM; ++i) acc[i] = 0.f;
      for (int k0 = 0; k0 < rep; k0 += kProjK) {
        const int kc = rep - k0 < kProjK ? rep - k0 : kProjK;
        __syncthreads();
        // stage rho[atom][k0 .. k0 + kc) transposed: coalesced along k, one atom per warp pass
        for (int at = warp; at < 32; at += kProjThreads / 32) {
          const long long aa = (long long)blockIdx.x * 32 + at;
          for (int k = lane; k < kc; k += 32) tile[k][at] = aa < n_atoms ? __ldg(rho + (size_t)aa * rep + k0 + k) : 0.f;
        }
        __syncthreads();
        if (mw == kProjM) proj_accumulate(acc, tile, kc, lane, Ue + (size_t)k0 * d + m0, d);
        else if (mw > 0) {
          for (int k = 0; k < kc; ++k) {
            const float av = tile[k][lane];
#pragma unroll
            for (int i = 0; i < kProjM; ++i)      // static indices: acc stays in registers
              if (i < mw) acc[i] = fmaf(__ldg(Ue + (size_t)(k0 + k) * d + m0 + i), av, acc[i]);
          }
        }
      }
      if (e_lane == e) {
#pragma unroll
        for (int i = 0; i < kProjM; ++i)
          if (i < mw) x[(size_t)a * d + m0 + i] = acc[i];
      }
    }
  }
}

// x, tiled: block = 64 consecutive atoms x 128 outputs, k in chunks of 16 through shared memory (rho transposed, U as is);
// thread = 4 atoms x 8 outputs (32 accumulators, 3 LDS.128 per 32 FMAs).  Atoms of different elements use different
// matrices: the block runs once per element present in its 64 atoms and keeps the rows of that element.  Used when
// d % 128 == 0 (the configs' d = 128 / 256); measured 15 625 atoms, rep 720, d 256: see DESIGN.md 5.5.
constexpr int kPxAtoms = 64, kPxOut = 128, kPxK = 16;
__global__ void __launch_bounds__(256)
project_x_tiled_kernel(const float* __restrict__ rho, const int32_t* __restrict__ elem, long long n_atoms, int rep, int d,
                       int n_elem, const float* __restrict__ U, float* __restrict__ x) {
  __shared__ __align__(16) float rt[kPxK][kPxAtoms + 4];     // rho^T chunk
  __shared__ __align__(16) float ut[kPxK][kPxOut];           // U chunk
  __shared__ int el[kPxAtoms];
  __shared__ int present[64];
  const int tid = threadIdx.x;
  const int ta = tid >> 4, tm = tid & 15;                    // 16 x 16 threads: atoms 4 ta .. +3, outputs 8 tm .. +7
  const long long a0 = (long long)blockIdx.x * kPxAtoms;
  const int m0 = blockIdx.y * kPxOut;
  if (tid < 64) present[tid] = 0;
  __syncthreads();
  if (tid < kPxAtoms) {
    const int e = a0 + tid < n_atoms ? __ldg(elem + a0 + tid) : -1;
    el[tid] = e;
    if (e >= 0) present[e & 63] = 1;
  }
  __syncthreads();
  for (int e = 0; e < n_elem; ++e) {
    if (n_elem <= 64 && !present[e]) continue;
    const float* Ue = U + (size_t)e * rep * d + m0;
    float acc[4][8];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 8; ++j) acc[i][j] = 0.f;
    for (int k0 = 0; k0 < rep; k0 += kPxK) {
      const int kc = rep - k0 < kPxK ? rep - k0 : kPxK;
      __syncthreads();
      // rho: 64 atoms x 16 k, thread = (atom tid / 4, 4 consecutive k); U: 16 k x 128 m, thread = (k tid / 16, 8 m)
      {
        const int at = tid >> 2, kq = (tid & 3) * 4;
        const bool ok = a0 + at < n_atoms && el[at] == e;
#pragma unroll
        for (int u = 0; u < 4; ++u)
          rt[kq + u][at] = (ok && kq + u < kc) ? __ldg(rho + (size_t)(a0 + at) * rep + k0 + kq + u) : 0.f;
        const int kk = tid >> 4, mq = (tid & 15) * 8;
        float4 u0 = make_float4(0.f, 0.f, 0.f, 0.f), u1 = u0;
        if (kk < kc) {
          u0 = __ldg(reinterpret_cast<const float4*>(Ue + (size_t)(k0 + kk) * d + mq));
          u1 = __ldg(reinterpret_cast<const float4*>(Ue + (size_t)(k0 + kk) * d + mq) + 1);
        }
        *reinterpret_cast<float4*>(&ut[kk][mq]) = u0;
        *reinterpret_cast<float4*>(&ut[kk][mq + 4]) = u1;
      }
      __syncthreads();
#pragma unroll
      for (int k = 0; k < kPxK; ++k) {
        const float4 r4 = *reinterpret_cast<const float4*>(&rt[k][4 * ta]);
        const float4 ua = *reinterpret_cast<const float4*>(&ut[k][8 * tm]);
        const float4 ub = *reinterpret_cast<const float4*>(&ut[k][8 * tm + 4]);
        const float rr[4] = {r4.x, r4.y, r4.z, r4.w};
        const float uu[8] = {ua.x, ua.y, ua.z, ua.w, ub.x, ub.y, ub.z, ub.w};
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 8; ++j) acc[i][j] = fmaf(rr[i], uu[j], acc[i][j]);
      }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int at = 4 * ta + i;
      if (a0 + at < n_atoms && el[at] == e) {
        float* dst = x + (size_t)(a0 + at) * d + m0 + 8 * tm;
        *reinterpret_cast<float4*>(dst) = make_float4(acc[i][0], acc[i][1], acc[i][2], acc[i][3]);
        *reinterpret_cast<float4*>(dst + 4) = make_float4(acc[i][4], acc[i][5], acc[i][6], acc[i][7]);
      }
    }
  }
}

// gradient: block = one atom I; its [rep][3n] block is projected to [d][3n], 32 columns at a time (lane = column).
__global__ void __launch_bounds__(kProjThreads)
project_grad_kernel(const float* __restrict__ gin, const int64_t* __restrict__ in_off, const int32_t* __restrict__ elem,
                    const int32_t* __restrict__ mol_off, int n_mol, int rep, int d, const float* __restrict__ U,
                    const int64_t* __restrict__ out_off, float* __restrict__ gout) {
  __shared__ float tile[kProjK][33];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int Ig = blockIdx.x;
  const int M = owner_molecule(mol_off, n_mol, Ig);
  const int a0 = __ldg(mol_off + M), n = __ldg(mol_off + M + 1) - a0, ncol = 3 * n;
  const float* src = gin + __ldg(in_off + M) + (size_t)(Ig - a0) * rep * ncol;    // [rep][ncol]
  float* dst = gout + __ldg(out_off + M) + (size_t)(Ig - a0) * d * ncol;           // [d][ncol]
  const float* Ue = U + (size_t)__ldg(elem + Ig) * rep * d;
  for (int c0 = 0; c0 < ncol; c0 += 32) {
    const int col = c0 + lane;
    for (int mp = 0; mp < d; mp += (kProjThreads / 32) * kProjM) {
      const int m0 = mp + warp * kProjM;
      const int mw = m0 >= d ? 0 : (d - m0 < kProjM ? d - m0 : kProjM);
      float acc[kProjM];
#pragma unroll
      for (int i = 0; i < kProjM; ++i) acc[i] = 0.f;
      for (int k0 = 0; k0 < rep; k0 += kProjK) {
        const int kc = rep - k0 < kProjK ? rep - k0 : kProjK;
        __syncthreads();
        for (int k = warp; k < kc; k += kProjThreads / 32)
          tile[k][lane] = col < ncol ? __ldg(src + (size_t)(k0 + k) * ncol + col) : 0.f;
        __syncthreads();
        if (mw == kProjM) proj_accumulate(acc, tile, kc, lane, Ue + (size_t)k0 * d + m0, d);
        else if (mw > 0) {
          for (int k = 0; k < kc; ++k) {
            const float av = tile[k][lane];
#pragma unroll
            for (int i = 0; i < kProjM; ++i)      // static indices: acc stays in registers
              if (i < mw) acc[i] = fmaf(__ldg(Ue + (size_t)(k0 + k) * d + m0 + i), av, acc[i]);
          }
        }
      }
      if (col < ncol) {
#pragma unroll
        for (int i = 0; i < kProjM; ++i)
          if (i < mw) dst[(size_t)(m0 + i) * ncol + col] = acc[i];
      }
    }
  }
}

// NEIGHBOR layout (the Jacobian of qmll_fchl19): block = one atom I; its S blocks [rep][3] are projected to [d][3], ten
// slots (30 columns, lane = (slot, c)) at a time.  Input chunks are staged with coalesced reads (a slot's [64 k][3] piece
// is 192 contiguous floats), outputs go through a per-warp shared-memory tile so that every slot's [32 m][3] piece is
// written as 96 contiguous floats.  Slots whose idx is negative are skipped (zero blocks).
// A Jacobian of FCHL19 is structurally sparse along k: the block of a neighbour of element Z_j is zero outside the
// two-body bin of Z_j and the pair bins that contain Z_j (n2 + 2 E n3 of E n2 + E (E + 1) n3 rows).  The slots are
// therefore taken in the order of their neighbour's element (so that the ten slots of a pass share their zero rows) and
// rows k whose 30 staged values are all zero are skipped (exact: they would add zeros): every lane tests two rows of the
// staged chunk, two ballots give the 64-bit mask of non-zero rows.
constexpr int kNbrSlots = 10;
constexpr int kNbrMaxS = 1024;     // slots that are reordered; beyond that the original order is kept

// 64-bit mask of the rows k of the staged chunk that hold a non-zero value (identical in every warp)
__device__ __forceinline__ unsigned long long proj_chunk_mask(const float (*tile)[33], int kc, int lane) {
  bool nz0 = false, nz1 = false;
  if (lane < kc) {
#pragma unroll 8
    for (int c = 0; c < 32; ++c) nz0 |= tile[lane][c] != 0.f;
  }
  if (lane + 32 < kc) {
#pragma unroll 8
    for (int c = 0; c < 32; ++c) nz1 |= tile[lane + 32][c] != 0.f;
  }
  return (unsigned long long)__ballot_sync(0xffffffffu, nz0) | ((unsigned long long)__ballot_sync(0xffffffffu, nz1) << 32);
}
__device__ __forceinline__ int nth_set_bit(unsigned long long m, int j) {
  const unsigned lo = (unsigned)m, hi = (unsigned)(m >> 32);
  const int c = __popc(lo);
  return j < c ? (int)__fns(lo, 0, j + 1) : 32 + (int)__fns(hi, 0, j - c + 1);
}
constexpr int kURow = (kProjThreads / 32) * kProjM;   // 256 columns of U per pass
constexpr int kUR = 32;                                // U rows staged at once (32 KB, shared with the output tiles)

__global__ void __launch_bounds__(kProjThreads)
project_nbr_kernel(const float* __restrict__ gin, const int32_t* __restrict__ idx, const int32_t* __restrict__ elem,
                   int S, int rep, int d, int n_elem, const float* __restrict__ U, float* __restrict__ gout) {
  __shared__ float tile[kProjK][33];
  __shared__ __align__(16) float otile[kProjThreads / 32][kProjM][33];
  float4* us4 = reinterpret_cast<float4*>(&otile[0][0][0]);       // [kUR][kURow] staged rows of U_e (kUR * kURow <= 8448)
  __shared__ short order[kNbrMaxS];      // live slots, grouped by the element of the slot's atom
  __shared__ int n_live_s;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const size_t I = blockIdx.x;
  const float* Ue = U + (size_t)__ldg(elem + I) * rep * d;
  // dead slots: zero blocks.  live slots: ordered by element (stable), by thread 0 of warp 0 with ballots per element
  if (warp == 0) {
    int n_live = 0;
    const int Sr = S < kNbrMaxS ? S : kNbrMaxS;
    for (int e = (idx ? 0 : n_elem - 1); e < n_elem; ++e)
      for (int base = 0; base < Sr; base += 32) {
        const int q = base + lane;
        bool take = false;
        if (q < Sr) {
          if (!idx) take = true;
          else {
            const int j = __ldg(idx + I * S + q);
            if (j >= 0) {
              int ej = __ldg(elem + j);
              ej = ej < 0 ? 0 : (ej >= n_elem ? n_elem - 1 : ej);
              take = ej == e;
            }
          }
        }
        const unsigned mask = __ballot_sync(0xffffffffu, take);
        if (take) order[n_live + __popc(mask & ((1u << lane) - 1u))] = (short)q;
        n_live += __popc(mask);
      }
    if (lane == 0) n_live_s = n_live;
  }
  __syncthreads();
  int n_live = n_live_s;
  if (idx) {
    for (int q = warp; q < S; q += kProjThreads / 32) {
      if (q < kNbrMaxS && __ldg(idx + I * S + q) >= 0) continue;
      if (q >= kNbrMaxS) continue;
      float* dst = gout + (I * S + q) * (size_t)d * 3;
      for (int t = lane; t < d * 3; t += 32) dst[t] = 0.f;
    }
  }
  const int n_total = n_live + (S > kNbrMaxS ? S - kNbrMaxS : 0);       // slots beyond the reorder window: as they are
  for (int q0 = 0; q0 < n_total; q0 += kNbrSlots) {
    const int nq = n_total - q0 < kNbrSlots ? n_total - q0 : kNbrSlots;
    auto slot_of = [&](int ql) { const int t = q0 + ql; return t < n_live ? (int)order[t] : kNbrMaxS + (t - n_live); };
    for (int mp = 0; mp < d; mp += (kProjThreads / 32) * kProjM) {
      const int m0 = mp + warp * kProjM;
      const int mw = m0 >= d ? 0 : (d - m0 < kProjM ? d - m0 : kProjM);
      float acc[kProjM];
#pragma unroll
      for (int i = 0; i < kProjM; ++i) acc[i] = 0.f;
      for (int k0 = 0; k0 < rep; k0 += kProjK) {
        const int kc = rep - k0 < kProjK ? rep - k0 : kProjK;
        __syncthreads();
        for (int ql = warp; ql < kNbrSlots + 1; ql += kProjThreads / 32) {   // warp = slot: no runtime division
          if (ql < nq) {
            const float* src = gin + ((I * S + slot_of(ql)) * rep + k0) * 3;
            for (int rem = lane; rem < kc * 3; rem += 32) {
              const int k = rem / 3;
              tile[k][ql * 3 + (rem - 3 * k)] = __ldcs(src + rem);
            }
          } else {                                                            // unused columns read as zeros
            const int c0 = ql < kNbrSlots ? ql * 3 : 30, c1 = ql < kNbrSlots ? c0 + 3 : 32;
            for (int k = lane; k < kc; k += 32)
              for (int c = c0; c < c1; ++c) tile[k][c] = 0.f;
          }
        }
        __syncthreads();
        // Non-zero rows of the chunk (the same mask in every warp).  Their U rows are staged in shared memory by the
        // whole block -- every load of a group of up to kUR rows is in flight at once -- and then read as broadcasts
        // (loading them row by row behind the zero test left the warps waiting on L2: 47 % long-scoreboard stalls).
        const unsigned long long mask = proj_chunk_mask(tile, kc, lane);
        const int nz = __popcll(mask);
        const int mlen = d - mp < kURow ? d - mp : kURow, m4 = mlen >> 2;     // columns of this pass (multiple of 4)
        unsigned long long rest = mask;
        for (int g0 = 0; g0 < nz; g0 += kUR) {
          const int ng = nz - g0 < kUR ? nz - g0 : kUR;
          if (g0 > 0) __syncthreads();                                        // the previous group has been consumed
          for (int item = threadIdx.x; item < ng * m4; item += kProjThreads) {
            const int jj = item / m4, c4 = item - jj * m4;
            const int k = nth_set_bit(mask, g0 + jj);
            us4[jj * (kURow / 4) + c4] = __ldg(reinterpret_cast<const float4*>(Ue + (size_t)(k0 + k) * d + mp) + c4);
          }
          __syncthreads();
          for (int jj = 0; jj < ng; ++jj) {
            const int k = __ffsll((long long)rest) - 1;
            rest &= rest - 1;
            if (mw > 0) {
              const float a = tile[k][lane];
              const float4* u4 = us4 + jj * (kURow / 4) + warp * (kProjM / 4);
#pragma unroll
              for (int q = 0; q < kProjM / 4; ++q) {
                if (4 * q < mw) {
                  const float4 u = u4[q];
                  acc[4 * q + 0] = fmaf(u.x, a, acc[4 * q + 0]);
                  if (4 * q + 1 < mw) acc[4 * q + 1] = fmaf(u.y, a, acc[4 * q + 1]);
                  if (4 * q + 2 < mw) acc[4 * q + 2] = fmaf(u.z, a, acc[4 * q + 2]);
                  if (4 * q + 3 < mw) acc[4 * q + 3] = fmaf(u.w, a, acc[4 * q + 3]);
                }
              }
            }
          }
        }
      }
      __syncthreads();      // the staged U rows share their storage with the output tiles
      // transpose through shared memory: slot ql gets [mw][3] contiguous floats at ((I S + q) d + m0) * 3
#pragma unroll
      for (int i = 0; i < kProjM; ++i) otile[warp][i][lane] = acc[i];
      __syncwarp();
      for (int ql = 0; ql < nq; ++ql) {
        float* dst = gout + ((I * S + slot_of(ql)) * (size_t)d + m0) * 3;
        for (int t = lane; t < mw * 3; t += 32) dst[t] = otile[warp][t / 3][ql * 3 + t % 3];
      }
      __syncwarp();
    }
  }
}

// Transposed projection (backward pass of x = rho^T U_e): w[I, k] = sum_m U[e_I, k, m] g[I, m].  Block = one atom, g in
// shared memory, one warp per row k of U_e (coalesced along m, shuffle reduction).
__global__ void __launch_bounds__(kProjThreads)
project_back_kernel(const float* __restrict__ g, const int32_t* __restrict__ elem, int rep, int d,
                    const float* __restrict__ U, float* __restrict__ w) {
  extern __shared__ float gs[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const size_t I = blockIdx.x;
  for (int m = threadIdx.x; m < d; m += kProjThreads) gs[m] = __ldg(g + I * d + m);
  __syncthreads();
  const float* Ue = U + (size_t)__ldg(elem + I) * rep * d;
  for (int k = warp; k < rep; k += kProjThreads / 32) {
    float acc = 0.f;
    for (int m = 4 * lane; m < d; m += 128) {
      const float4 u = __ldg(reinterpret_cast<const float4*>(Ue + (size_t)k * d + m));
      acc = fmaf(u.x, gs[m], acc); acc = fmaf(u.y, gs[m + 1], acc);
      acc = fmaf(u.z, gs[m + 2], acc); acc = fmaf(u.w, gs[m + 3], acc);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) w[I * rep + k] = acc;
  }
}

// The same product tiled like project_x_tiled_kernel: block = 64 atoms x 128 rows k of U_e, the contraction index m in
// chunks of 16 (g transposed and U^T in shared memory), thread = 4 atoms x 8 rows; once per element present in the block.
__global__ void __launch_bounds__(256)
project_back_tiled_kernel(const float* __restrict__ g, const int32_t* __restrict__ elem, long long n_atoms, int rep, int d,
                          int n_elem, const float* __restrict__ U, float* __restrict__ w) {
  __shared__ __align__(16) float gt[kPxK][kPxAtoms + 4];     // g^T chunk
  __shared__ __align__(16) float ut[kPxK][kPxOut + 4];       // U^T chunk: [m][row k]
  __shared__ int el[kPxAtoms];
  __shared__ int present[64];
  const int tid = threadIdx.x;
  const int ta = tid >> 4, tm = tid & 15;
  const long long a0 = (long long)blockIdx.x * kPxAtoms;
  const int r0 = blockIdx.y * kPxOut;
  if (tid < 64) present[tid] = 0;
  __syncthreads();
  if (tid < kPxAtoms) {
    const int e = a0 + tid < n_atoms ? __ldg(elem + a0 + tid) : -1;
    el[tid] = e;
    if (e >= 0) present[e & 63] = 1;
  }
  __syncthreads();
  for (int e = 0; e < n_elem; ++e) {
    if (n_elem <= 64 && !present[e]) continue;
    const float* Ue = U + (size_t)e * rep * d;
    float acc[4][8];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 8; ++j) acc[i][j] = 0.f;
    for (int m0 = 0; m0 < d; m0 += kPxK) {          // d is a multiple of 16 here
      __syncthreads();
      {
        const int at = tid >> 2, mq = (tid & 3) * 4;
        const bool ok = a0 + at < n_atoms && el[at] == e;
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        if (ok) v = __ldg(reinterpret_cast<const float4*>(g + (size_t)(a0 + at) * d + m0 + mq));
        gt[mq][at] = v.x; gt[mq + 1][at] = v.y; gt[mq + 2][at] = v.z; gt[mq + 3][at] = v.w;
        const int rr = tid >> 1, mh = (tid & 1) * 8;      // row r0 + rr of U_e, 8 consecutive m
        float4 u0 = make_float4(0.f, 0.f, 0.f, 0.f), u1 = u0;
        if (r0 + rr < rep) {
          const float4* src = reinterpret_cast<const float4*>(Ue + (size_t)(r0 + rr) * d + m0 + mh);
          u0 = __ldg(src); u1 = __ldg(src + 1);
        }
        ut[mh][rr] = u0.x; ut[mh + 1][rr] = u0.y; ut[mh + 2][rr] = u0.z; ut[mh + 3][rr] = u0.w;
        ut[mh + 4][rr] = u1.x; ut[mh + 5][rr] = u1.y; ut[mh + 6][rr] = u1.z; ut[mh + 7][rr] = u1.w;
      }
      __syncthreads();
#pragma unroll
      for (int k = 0; k < kPxK; ++k) {
        const float4 r4 = *reinterpret_cast<const float4*>(&gt[k][4 * ta]);
        const float4 ua = *reinterpret_cast<const float4*>(&ut[k][8 * tm]);
        const float4 ub = *reinterpret_cast<const float4*>(&ut[k][8 * tm + 4]);
        const float rr[4] = {r4.x, r4.y, r4.z, r4.w};
        const float uu[8] = {ua.x, ua.y, ua.z, ua.w, ub.x, ub.y, ub.z, ub.w};
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 8; ++j) acc[i][j] = fmaf(rr[i], uu[j], acc[i][j]);
      }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int at = 4 * ta + i;
      if (a0 + at < n_atoms && el[at] == e) {
#pragma unroll
        for (int j = 0; j < 8; ++j)
          if (r0 + 8 * tm + j < rep) w[(size_t)(a0 + at) * rep + r0 + 8 * tm + j] = acc[i][j];
      }
    }
  }
}

int project_back_launch(const float* g, const int32_t* elem, int64_t n_atoms, int32_t rep, int32_t d, int32_t n_elem,
                        const float* U, float* w, cudaStream_t st) {
  if (n_atoms == 0) return QMLL_OK;
  if (d % kPxK == 0) {
    dim3 grid((unsigned)((n_atoms + kPxAtoms - 1) / kPxAtoms), (unsigned)((rep + kPxOut - 1) / kPxOut));
    project_back_tiled_kernel<<<grid, 256, 0, st>>>(g, elem, n_atoms, rep, d, n_elem, U, w);
    QMLL_LAUNCH_CHECK("project_back_tiled_kernel");
    return QMLL_OK;
  }
  project_back_kernel<<<(unsigned)n_atoms, kProjThreads, d * sizeof(float), st>>>(g, elem, rep, d, U, w);
  QMLL_LAUNCH_CHECK("project_back_kernel");
  return QMLL_OK;
}

int project_neighbor_launch(const float* gin, const int32_t* idx, const int32_t* elem, int64_t n_atoms, int32_t S,
                            int32_t rep, int32_t d, int32_t n_elem, const float* U, float* gout, cudaStream_t st) {
  if (n_atoms == 0 || S == 0) return QMLL_OK;
  project_nbr_kernel<<<(unsigned)n_atoms, kProjThreads, 0, st>>>(gin, idx, elem, S, rep, d, n_elem, U, gout);
  QMLL_LAUNCH_CHECK("project_nbr_kernel");
  return QMLL_OK;
}

int project_launch(const float* rho, const int32_t* elem, const int32_t* mol_off, int64_t n_atoms, int32_t n_mol,
                   int32_t rep, int32_t d, int32_t n_elem, const float* U, float* x, const float* gin,
                   const int64_t* in_off, float* gout, const int64_t* out_off, cudaStream_t st) {
  if (n_atoms == 0) return QMLL_OK;
  if (x) {
    if (d % kPxOut == 0) {
      dim3 grid((unsigned)((n_atoms + kPxAtoms - 1) / kPxAtoms), (unsigned)(d / kPxOut));
      project_x_tiled_kernel<<<grid, 256, 0, st>>>(rho, elem, n_atoms, rep, d, n_elem, U, x);
      QMLL_LAUNCH_CHECK("project_x_tiled_kernel");
    } else {
      project_x_kernel<<<(unsigned)((n_atoms + 31) / 32), kProjThreads, 0, st>>>(rho, elem, n_atoms, rep, d, n_elem, U, x);
      QMLL_LAUNCH_CHECK("project_x_kernel");
    }
  }
  if (gout) {
    project_grad_kernel<<<(unsigned)n_atoms, kProjThreads, 0, st>>>(gin, in_off, elem, mol_off, n_mol, rep, d, U,
                                                                   out_off, gout);
    QMLL_LAUNCH_CHECK("project_grad_kernel");
  }
  return QMLL_OK;
}

}  // namespace qmll
