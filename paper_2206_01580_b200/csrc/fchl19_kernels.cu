// fchl19_kernels.cu -- NEXT row f3 of SURVEY.md section 8(f): the FCHL19 atomic representation (PAPER.md section E,
// eq. 23-33) and its Jacobian with respect to the atomic positions, in the neighbour-sparse layout that
// qmll_project_neighbor / qmll_predict / qmll_sorf_forward consume (qmll_grad NEIGHBOR).
//
//   two-body  (eq. 24-27):  rho_i[X, s]        = sum_{j: Z_j = X} f(r_ij) r_ij^-N2 LogNormal(R_s; mu(r_ij), sigma(r_ij))
//   three-body (eq. 28-33): rho_i[{X,Y}, s, a] = sum_{j<k: {Z_j,Z_k} = {X,Y}} xi_3 Radial_s((r_ij + r_ik)/2) Ang_a(theta_i)
//                                                 f(r_ij) f(r_ik) f(r_jk)
// Readings B1-B9 of DESIGN.md (grids, cut-off, three cut-offs, unordered pairs, layout) are the oracle's.
//
// Design (the paper's: one block per atom, 16 x 8 threads over (j, k), reduction in global memory, L246-268).  Here:
// one block per atom, neighbours inside r_cut compacted and sorted by element in shared memory, and then one WARP
// per neighbour slot j:
//   * the lanes first run over the partners k and store the s-independent part of every (j, k) term and of its
//     gradient with respect to r_j (12 floats) in a per-warp shared-memory table -- all the transcendental and
//     vector work, done once per pair and not once per radial grid point;
//   * then lane = radial grid point s: for every element pair bin that contains Z_j the lane runs over the partners
//     of the other element (contiguous after the sort) and needs one exp and 10 FMAs per partner;
//   * the [rep, 3] Jacobian block of the slot is written exactly once, coalesced, zeros included (no memset pass, no
//     global atomics); the block of the central atom is minus the sum of the others (translation invariance) and is
//     accumulated in shared memory.
// The Jacobian is the big output: (K + 1) rep 3 floats per atom (15 625-atom cell, K = 64: 8.8 GB).  Measured
// (profiles/r2_fchl19_featmap.md): 2.9 ms = 3.0 TB/s of writes (0.46 of the HBM copy peak) at 32 warps / SM (four
// blocks: tables sized by K, 64 registers) -- issue-bound (~170 k warp instructions per atom), not yet write-bound;
// 3.9 ms with two blocks per SM.
// Mode 2 (qmll_fchl19_backward) is the Jacobian-free backward pass: the same loops, but every lane multiplies what it
// would have written by dE/d rho and the warp reduces to one force vector per neighbour (1.65 ms, nothing materialised).
#include <math_constants.h>

#include "qmll_common.cuh"

namespace qmll {

constexpr int kFchlThreads = 256;
constexpr int kFchlWarps = kFchlThreads / 32;
constexpr int kFchlMaxN = QMLL_FCHL19_MAX_NEIGHBOURS;   // neighbours inside r_cut per atom
constexpr int kPairF = 12;                              // floats per (j, k) table entry
constexpr int kFchlMaxElem = 16;

struct FchlDev {
  int E, n2, n3, rep, K;
  int cap;                            // rows of the shared-memory neighbour tables: min(K rounded up to 4, kFchlMaxN)
  float eta2, eta3, N2, N3, c3d;      // c3d = c3 * 2 exp(-zeta^2 / 2)   (n = 1 Fourier terms, reading B5)
  float rcut, inv_rcut, rs2_step, rs3_step, norm3;
};

struct FchlSmem {
  float *vx, *vy, *vz, *rr, *fc, *dfc;   // [cap] sorted neighbour table: vector i -> j, length, f, f'
  int *ne, *nslot;                       // [cap] element, neighbour slot q
  int* e_start;                          // [kFchlMaxElem + 1] first sorted index of every element
  int* misc;                             // [4]: nn, n_invalid
  int* inv_list;                         // [K] slots that hold no neighbour inside r_cut
  float* rho_acc;                        // [rep]
  float* self_acc;                       // [3 rep]
  float* pair_tab;                       // [warps][cap][kPairF]
  float* stage;                          // [warps][192]
};

// The tables hold `cap` neighbours: no more than K slots can be inside r_cut, so K (not the library-wide maximum) sizes
// them -- 36 KB instead of 76 KB per block at K = 64, which is what lets 4-5 blocks share an SM.
__host__ __device__ inline int fchl_cap(int K) {
  const int k4 = (K + 3) & ~3;
  return k4 < 4 ? 4 : (k4 > kFchlMaxN ? kFchlMaxN : k4);
}
__host__ __device__ inline size_t fchl_smem_floats(int rep, int K, bool jac) {
  const size_t cap = (size_t)fchl_cap(K);
  return 8 * cap + 32 + 8 + (size_t)K + (size_t)rep + (jac ? (size_t)3 * rep : 0) + (size_t)kFchlWarps * cap * kPairF +
         (size_t)kFchlWarps * 192 + 16;
}

__device__ __forceinline__ FchlSmem fchl_carve(float* sm, int rep, int K, int cap, bool jac) {
  FchlSmem s;
  s.pair_tab = sm;  sm += kFchlWarps * cap * kPairF;            // first: 16-byte aligned float4 rows
  s.stage = sm;     sm += kFchlWarps * 192;
  s.vx = sm; s.vy = sm + cap; s.vz = sm + 2 * cap; s.rr = sm + 3 * cap;
  s.fc = sm + 4 * cap; s.dfc = sm + 5 * cap;
  s.ne = reinterpret_cast<int*>(sm + 6 * cap);
  s.nslot = s.ne + cap;
  s.e_start = s.nslot + cap;
  s.misc = s.e_start + 32;
  s.inv_list = s.misc + 8;
  s.rho_acc = reinterpret_cast<float*>(s.inv_list + K);
  s.self_acc = s.rho_acc + rep;
  return s;
}

// f_cut and its derivative (eq. 27), r < r_cut
__device__ __forceinline__ void f_cut_pair(float r, const FchlDev& P, float* f, float* df) {
  float sn, cs;
  sincospif(r * P.inv_rcut, &sn, &cs);
  *f = 0.5f * (cs + 1.f);
  *df = -0.5f * CUDART_PI_F * P.inv_rcut * sn;
}

// kMode 0: representation only; 1: + Jacobian blocks; 2: vector-Jacobian product (backward pass, L268: "the force
// components are stored and summed in on-chip memory"): F[j] -= sum_k w_i[k] d rho_i[k] / d r_j for every neighbour
// image j, F[i] += the same sum (translation invariance), with w_i = dE / d rho_i given -- no Jacobian is materialised.
template <int kMode>
__global__ void __launch_bounds__(kFchlThreads, kMode == 0 ? 5 : 4)
fchl19_kernel(const FchlDev P, const float* __restrict__ r, const int32_t* __restrict__ elem,
              const int32_t* __restrict__ nbr_idx, const float* __restrict__ nbr_shift, long long n_atoms,
              float* __restrict__ rho, int32_t* __restrict__ jac_idx, float* __restrict__ jac_val,
              int32_t* __restrict__ info, const float* __restrict__ w_in, float* __restrict__ forces) {
  constexpr bool kJac = kMode == 1, kVjp = kMode == 2, kGrad = kMode != 0;
  extern __shared__ __align__(16) float sm_raw[];
  const FchlSmem S = fchl_carve(sm_raw, P.rep, P.K, P.cap, kGrad);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long i = blockIdx.x;
  const int rep = P.rep, K = P.K, off3 = P.E * P.n2;
  const float rix = __ldg(r + 3 * i), riy = __ldg(r + 3 * i + 1), riz = __ldg(r + 3 * i + 2);

  for (int t = threadIdx.x; t < rep * (kJac ? 4 : 1); t += kFchlThreads) S.rho_acc[t] = 0.f;   // rho_acc + self_acc
  if (kVjp)                                                                                    // w_i in place of self_acc
    for (int t = threadIdx.x; t < rep; t += kFchlThreads) S.self_acc[t] = __ldg(w_in + (size_t)i * rep + t);

  // ---- phase 0a: warp 0 compacts the neighbours inside r_cut (in slot order: deterministic) ----
  if (warp == 0) {
    int cnt = 0, n_inv = 0;
    for (int base = 0; base < K; base += 32) {
      const int q = base + lane;
      int j = -1;
      float dx = 0.f, dy = 0.f, dz = 0.f, d2 = 0.f;
      if (q < K) j = __ldg(nbr_idx + i * K + q);
      if (j >= 0) {
        dx = __ldg(r + 3 * (size_t)j) - rix; dy = __ldg(r + 3 * (size_t)j + 1) - riy; dz = __ldg(r + 3 * (size_t)j + 2) - riz;
        if (nbr_shift) {
          const float* sh = nbr_shift + ((size_t)i * K + q) * 3;
          dx += __ldg(sh); dy += __ldg(sh + 1); dz += __ldg(sh + 2);
        }
        d2 = dx * dx + dy * dy + dz * dz;
      }
      const bool valid = j >= 0 && d2 < P.rcut * P.rcut && d2 > 0.f;
      const unsigned mask = __ballot_sync(0xffffffffu, valid);
      const unsigned imask = __ballot_sync(0xffffffffu, q < K && !valid);
      const unsigned lt = (1u << lane) - 1u;
      const int pos = cnt + __popc(mask & lt);
      if (valid && pos < P.cap) {
        S.vx[pos] = dx; S.vy[pos] = dy; S.vz[pos] = dz; S.rr[pos] = sqrtf(d2);
        S.ne[pos] = __ldg(elem + j); S.nslot[pos] = kVjp ? j : q;     // backward: the atom that receives the force
      }
      if (q < K && !valid) S.inv_list[n_inv + __popc(imask & lt)] = q;
      if (kJac && q < K) jac_idx[i * (K + 1) + 1 + q] = (valid && pos < P.cap) ? j : -1;
      cnt += __popc(mask);
      n_inv += __popc(imask);
    }
    if (lane == 0) {
      if (cnt > P.cap) { atomicMax(info, (int)(i < 0x7fffffff ? i + 1 : 0x7fffffff)); cnt = P.cap; }
      S.misc[0] = cnt; S.misc[1] = n_inv;
      if (kJac) jac_idx[i * (K + 1)] = (int32_t)i;
    }
  }
  __syncthreads();
  const int nn = S.misc[0], n_inv = S.misc[1];

  // ---- phase 0b: stable counting sort by element, cut-off values ----
  {
    float ex = 0.f, ey = 0.f, ez = 0.f, er = 1.f;
    int ee = 0, es = 0, pos = 0;
    const int m = threadIdx.x;
    if (m < nn) {
      ex = S.vx[m]; ey = S.vy[m]; ez = S.vz[m]; er = S.rr[m]; ee = S.ne[m]; es = S.nslot[m];
      for (int t = 0; t < nn; ++t) {
        const int et = S.ne[t];
        pos += (et < ee || (et == ee && t < m)) ? 1 : 0;
      }
    }
    if (m <= P.E) {
      int c = 0;
      for (int t = 0; t < nn; ++t) c += (S.ne[t] < m) ? 1 : 0;
      S.e_start[m] = c;
    }
    __syncthreads();
    if (m < nn) {
      float f, df;
      f_cut_pair(er, P, &f, &df);
      S.vx[pos] = ex; S.vy[pos] = ey; S.vz[pos] = ez; S.rr[pos] = er; S.fc[pos] = f; S.dfc[pos] = df;
      S.ne[pos] = ee; S.nslot[pos] = es;
    }
    __syncthreads();
  }

  // slots without a neighbour: zero Jacobian blocks
  if (kJac) {
    for (int t = 0; t < n_inv; ++t) {
      float* jb = jac_val + ((size_t)i * (K + 1) + 1 + S.inv_list[t]) * (size_t)rep * 3;
      for (int u = threadIdx.x; u < rep * 3; u += kFchlThreads) jb[u] = 0.f;
    }
  }

  // ---- phase 1: one warp per neighbour slot ----
  float* pt = S.pair_tab + warp * (P.cap * kPairF);
  float* stage = S.stage + warp * 192;
  const float* wv = S.self_acc;                 // kVjp: dE / d rho_i
  float self_x = 0.f, self_y = 0.f, self_z = 0.f;
  for (int m = warp; m < nn; m += kFchlWarps) {
    float fx = 0.f, fy = 0.f, fz = 0.f;         // kVjp: sum_k w[k] d rho_i[k] / d r_j, per lane
    const float ax = S.vx[m], ay = S.vy[m], az = S.vz[m], ra = S.rr[m], Fa = S.fc[m], dFa = S.dfc[m];
    const float ira = 1.f / ra, hx = ax * ira, hy = ay * ira, hz = az * ira;     // unit vector i -> j
    const int Zj = S.ne[m];
    float* jb = kJac ? jac_val + ((size_t)i * (K + 1) + 1 + S.nslot[m]) * (size_t)rep * 3 : nullptr;

    // (a) two-body term of j and d/dr_j of it (eq. 24-26): lane = grid point s
    {
      const float r2 = ra * ra;
      const float sig2 = log1pf(P.eta2 / r2);                     // eq. 26
      const float mu = logf(ra) - 0.5f * sig2;                    // eq. 25
      const float dsig2 = -2.f * P.eta2 / (ra * (r2 + P.eta2));
      const float dmu = ira - 0.5f * dsig2;
      const float rpw = expf(-P.N2 * logf(ra));
      float dg = 0.f;
      if (lane < P.n2) {
        const float Rs = P.rs2_step * (float)(lane + 1);
        const float t = logf(Rs) - mu;
        const float L = expf(-t * t / (2.f * sig2)) / (Rs * sqrtf(sig2) * 2.5066282746310002f);
        atomicAdd(&S.rho_acc[Zj * P.n2 + lane], Fa * rpw * L);
        const float dlnL = (-0.5f * dsig2 + t * dmu + 0.5f * t * t * dsig2 / sig2) / sig2;
        dg = rpw * L * (dFa + Fa * (dlnL - P.N2 * ira));
      }
      if (kVjp && lane < P.n2) {
        const float t = wv[Zj * P.n2 + lane] * dg;
        fx = t * hx; fy = t * hy; fz = t * hz;
      }
      if (kJac) {
        if (lane < P.n2) { stage[3 * lane] = dg * hx; stage[3 * lane + 1] = dg * hy; stage[3 * lane + 2] = dg * hz; }
        __syncwarp();
        for (int X = 0; X < P.E; ++X)
          for (int t = lane; t < 3 * P.n2; t += 32) {
            const float v = X == Zj ? stage[t] : 0.f;
            jb[X * P.n2 * 3 + t] = v;
            if (X == Zj) atomicAdd(&S.self_acc[X * P.n2 * 3 + t], -v);
          }
        __syncwarp();
      }
    }

    // (b) per-partner table: the part of every (j, k) term that does not depend on the radial grid point
    for (int kk = lane; kk < nn; kk += 32) {
      float4 o0 = make_float4(0.f, 0.f, 0.f, 0.f), o1 = o0, o2 = o0;
      if (kk != m) {
        const float bx = S.vx[kk], by = S.vy[kk], bz = S.vz[kk], rb = S.rr[kk], Fb = S.fc[kk];
        const float cx = bx - ax, cy = by - ay, cz = bz - az;
        const float rc2 = cx * cx + cy * cy + cz * cz;
        if (rc2 < P.rcut * P.rcut && rc2 > 0.f) {                  // third cut-off, reading B3
          const float rc = sqrtf(rc2), irc = 1.f / rc, irb = 1.f / rb;
          const float gx = bx * irb, gy = by * irb, gz = bz * irb;     // unit i -> k
          const float ux = cx * irc, uy = cy * irc, uz = cz * irc;     // unit j -> k
          float Fc, dFc;
          f_cut_pair(rc, P, &Fc, &dFc);
          const float cosi = hx * gx + hy * gy + hz * gz;              // angle at i
          const float cosj = -(hx * ux + hy * uy + hz * uz);           // angle at j
          const float cosk = gx * ux + gy * uy + gz * uz;              // angle at k
          const float wx = hy * gz - hz * gy, wy = hz * gx - hx * gz, wz = hx * gy - hy * gx;
          const float sini = sqrtf(wx * wx + wy * wy + wz * wz);
          const float Nn = 1.f + 3.f * cosi * cosj * cosk;             // eq. 30 numerator
          const float Dn = expf(-P.N3 * logf(ra * rb * rc));           // (r_ij r_ik r_jk)^-N3
          const float FF = Fa * Fb * Fc;
          const float Pv = P.c3d * Nn * Dn * FF;
          o1.z = Pv * cosi; o1.w = Pv * sini; o2.x = 0.5f * (ra + rb);
          if (kGrad) {
            // gradients with respect to the position of j
            const float ci_x = (gx - cosi * hx) * ira, ci_y = (gy - cosi * hy) * ira, ci_z = (gz - cosi * hz) * ira;
            const float cj_x = -((ux + cosj * hx) * ira - (hx + cosj * ux) * irc);
            const float cj_y = -((uy + cosj * hy) * ira - (hy + cosj * uy) * irc);
            const float cj_z = -((uz + cosj * hz) * ira - (hz + cosj * uz) * irc);
            const float ck_x = -(gx - cosk * ux) * irc, ck_y = -(gy - cosk * uy) * irc, ck_z = -(gz - cosk * uz) * irc;
            const float a1 = 3.f * cosj * cosk, a2 = 3.f * cosi * cosk, a3 = 3.f * cosi * cosj;
            const float nx = a1 * ci_x + a2 * cj_x + a3 * ck_x;
            const float ny = a1 * ci_y + a2 * cj_y + a3 * ck_y;
            const float nz = a1 * ci_z + a2 * cj_z + a3 * ck_z;
            // P = c3d N D Fa Fb Fc:  grad P = c3d D Fb [ gradN Fa Fc + N (-N3)(h/ra - u/rc) Fa Fc + N (Fa' Fc h - Fa Fc' u) ]
            const float ka = Nn * (dFa * Fc - P.N3 * ira * Fa * Fc);       // coefficient of h
            const float kc = Nn * (-Fa * dFc + P.N3 * irc * Fa * Fc);      // coefficient of u
            const float pre = P.c3d * Dn * Fb, FaFc = Fa * Fc;
            const float px = pre * (nx * FaFc + ka * hx + kc * ux);
            const float py = pre * (ny * FaFc + ka * hy + kc * uy);
            const float pz = pre * (nz * FaFc + ka * hz + kc * uz);
            const float ct = -cosi / fmaxf(sini, 1e-6f);                   // d sin / d cos (collinear: clamped)
            o0.x = px * cosi + Pv * ci_x; o0.y = py * cosi + Pv * ci_y; o0.z = pz * cosi + Pv * ci_z;
            o0.w = px * sini + Pv * ct * ci_x; o1.x = py * sini + Pv * ct * ci_y; o1.y = pz * sini + Pv * ct * ci_z;
          }
        }
      }
      float4* dst = reinterpret_cast<float4*>(pt + kk * kPairF);
      dst[0] = o0; dst[1] = o1; dst[2] = o2;
    }
    __syncwarp();

    // (c) lane = radial grid point s of the three-body term; bins (X <= Y) in the order of reading B7
    const float Rs = P.rs3_step * (float)(lane + 1);
    int p = 0;
    for (int X = 0; X < P.E; ++X)
      for (int Y = X; Y < P.E; ++Y, ++p) {
        const bool hit = X == Zj || Y == Zj;
        const int base = (off3 + p * P.n3 * 2) * 3;
        if (!hit) {
          if (kJac)
            for (int t = lane; t < 6 * P.n3; t += 32) jb[base + t] = 0.f;
          continue;
        }
        const int other = X == Zj ? Y : X;
        const int k0 = S.e_start[other], k1 = S.e_start[other + 1];
        float acx = 0.f, acy = 0.f, acz = 0.f, bc = 0.f, asx = 0.f, asy = 0.f, asz = 0.f, bs = 0.f, vc = 0.f, vs = 0.f;
        if (lane < P.n3) {
          for (int kk = k0; kk < k1; ++kk) {
            const float4* q = reinterpret_cast<const float4*>(pt + kk * kPairF);
            const float4 q0 = q[0], q1 = q[1];
            const float dm = q[2].x - Rs;
            const float R = P.norm3 * __expf(-P.eta3 * dm * dm);          // eq. 29
            if (kGrad) {
              const float w = -P.eta3 * dm * R;                            // dR/dm * dm/dr_ij, times h below
              acx = fmaf(R, q0.x, acx); acy = fmaf(R, q0.y, acy); acz = fmaf(R, q0.z, acz); bc = fmaf(w, q1.z, bc);
              asx = fmaf(R, q0.w, asx); asy = fmaf(R, q1.x, asy); asz = fmaf(R, q1.y, asz); bs = fmaf(w, q1.w, bs);
            }
            if (kk > m) { vc = fmaf(R, q1.z, vc); vs = fmaf(R, q1.w, vs); }   // every unordered pair once (B6)
          }
          if (k1 > k0 && !kVjp) {
            atomicAdd(&S.rho_acc[off3 + (p * P.n3 + lane) * 2], vc);
            atomicAdd(&S.rho_acc[off3 + (p * P.n3 + lane) * 2 + 1], vs);
          }
          if (kVjp && k1 > k0) {
            const float wc = wv[off3 + (p * P.n3 + lane) * 2], wsn = wv[off3 + (p * P.n3 + lane) * 2 + 1];
            fx += wc * (acx + bc * hx) + wsn * (asx + bs * hx);
            fy += wc * (acy + bc * hy) + wsn * (asy + bs * hy);
            fz += wc * (acz + bc * hz) + wsn * (asz + bs * hz);
          }
        }
        if (kJac) {
          if (lane < P.n3) {
            stage[6 * lane + 0] = acx + bc * hx; stage[6 * lane + 1] = acy + bc * hy; stage[6 * lane + 2] = acz + bc * hz;
            stage[6 * lane + 3] = asx + bs * hx; stage[6 * lane + 4] = asy + bs * hy; stage[6 * lane + 5] = asz + bs * hz;
          }
          __syncwarp();
          for (int t = lane; t < 6 * P.n3; t += 32) {
            const float v = stage[t];
            jb[base + t] = v;
            if (k1 > k0) atomicAdd(&S.self_acc[base + t], -v);
          }
          __syncwarp();
        }
      }
    if (kVjp) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        fx += __shfl_xor_sync(0xffffffffu, fx, o);
        fy += __shfl_xor_sync(0xffffffffu, fy, o);
        fz += __shfl_xor_sync(0xffffffffu, fz, o);
      }
      if (lane == 0) {
        float* Fj = forces + 3 * (size_t)S.nslot[m];
        atomicAdd(Fj, -fx); atomicAdd(Fj + 1, -fy); atomicAdd(Fj + 2, -fz);
      }
      self_x += fx; self_y += fy; self_z += fz;
    }
    __syncwarp();
  }
  if (kVjp && lane == 0 && (self_x != 0.f || self_y != 0.f || self_z != 0.f)) {
    float* Fi = forces + 3 * (size_t)i;
    atomicAdd(Fi, self_x); atomicAdd(Fi + 1, self_y); atomicAdd(Fi + 2, self_z);
  }
  __syncthreads();

  // ---- phase 2: results of the atom ----
  if (rho && !kVjp)
    for (int t = threadIdx.x; t < rep; t += kFchlThreads) rho[(size_t)i * rep + t] = S.rho_acc[t];
  if (kJac) {
    float* jb = jac_val + (size_t)i * (K + 1) * (size_t)rep * 3;
    for (int t = threadIdx.x; t < rep * 3; t += kFchlThreads) jb[t] = S.self_acc[t];
  }
}

int fchl19_rep_size(const qmll_fchl19_params* fp) { return fp->n_elem * fp->n2 + fp->n_elem * (fp->n_elem + 1) * fp->n3; }

int fchl19_launch(const qmll_fchl19_params* fp, const float* r, const int32_t* elem, int64_t n_atoms,
                  const int32_t* nbr_idx, const float* nbr_shift, int32_t K, float* rho, int32_t* jac_idx,
                  float* jac_val, int32_t* info, const float* w_in, float* forces, cudaStream_t st) {
  FchlDev P;
  P.E = fp->n_elem; P.n2 = fp->n2; P.n3 = fp->n3; P.rep = fchl19_rep_size(fp); P.K = K; P.cap = fchl_cap(K);
  P.eta2 = fp->eta2; P.eta3 = fp->eta3; P.N2 = fp->two_body_decay; P.N3 = fp->three_body_decay;
  P.c3d = (float)((double)fp->three_body_weight * 2.0 * exp(-0.5 * (double)fp->zeta * (double)fp->zeta));
  P.rcut = fp->r_cut; P.inv_rcut = 1.f / fp->r_cut;
  P.rs2_step = fp->r_cut / (float)fp->n2; P.rs3_step = fp->r_cut / (float)fp->n3;
  P.norm3 = (float)sqrt((double)fp->eta3 / 3.14159265358979323846);
  QMLL_CUDA_TRY(cudaMemsetAsync(info, 0, sizeof(int32_t), st));
  if (forces) QMLL_CUDA_TRY(cudaMemsetAsync(forces, 0, (size_t)n_atoms * 3 * sizeof(float), st));
  if (n_atoms == 0) return QMLL_OK;
  const int mode = forces ? 2 : (jac_val ? 1 : 0);
  const size_t smem = fchl_smem_floats(P.rep, K, mode != 0) * sizeof(float);
  if (smem > 227 * 1024) return QMLL_ERR_UNSUPPORTED;
  auto launch = [&](auto kern) -> int {
    QMLL_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<(unsigned)n_atoms, kFchlThreads, smem, st>>>(P, r, elem, nbr_idx, nbr_shift, n_atoms, rho, jac_idx, jac_val, info,
                                                        w_in, forces);
    return QMLL_OK;
  };
  int rc = mode == 2 ? launch(fchl19_kernel<2>) : (mode == 1 ? launch(fchl19_kernel<1>) : launch(fchl19_kernel<0>));
  if (rc) return rc;
  QMLL_LAUNCH_CHECK("fchl19_kernel");
  return QMLL_OK;
}

}  // namespace qmll
