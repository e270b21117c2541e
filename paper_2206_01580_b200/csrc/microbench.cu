// microbench.cu -- measures the roofline denominators MEASURED_PEAKS.json lacks:
// issue rates of the plain-ALU instructions the fused SORF kernels are bound by (FADD, FADD2 = add.f32x2, FFMA,
// LOP3, SHF, mixes of them, MUFU.COS, SHFL) and the shared-memory load bandwidth.  Each kernel runs a register-only
// loop of independent dependency chains on every SM and reports BOTH lane-operations per SM clock (from clock64,
// independent of DVFS) and wall time (CUDA events, by the caller), so a roofline can be stated at the clock the
// product kernels actually ran at.  Not on the product path; called by paper_2206_01580_b200/peaks.py.
#include <stdint.h>

#include "qmll_common.cuh"
#include "tcgen05_utils.cuh"

namespace qmll {

constexpr int kMbThreads = 256;
constexpr int kMbUnroll = 16;   // independent chains per thread

enum MbKind {
  kMbFadd = 0, kMbFfma = 1, kMbFadd2 = 2, kMbFfma2 = 3, kMbLop3 = 4, kMbShf = 5, kMbFadd2Lop3 = 6,
  kMbFaddSign = 7, kMbFadd2Sign = 8, kMbMufuCos = 9, kMbLds128 = 10, kMbShfl = 11, kMbFadd2Lop3Shf = 12,
  kMbDfma = 13, kMbDmma = 14,   // FP64: scalar DFMA, mma.sync.m8n8k4.f64 (the solve's trailing update)
  kMbCount = 15
};

__device__ __forceinline__ uint64_t pack2(float a, float b) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
  return r;
}
__device__ __forceinline__ float lo_of(uint64_t v) {
  float a, b;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
  return a + b;
}

// One kernel per instruction mix; `ops` counted per thread and iteration is returned by mb_ops_per_iter().
template <int KIND>
__global__ void __launch_bounds__(kMbThreads)
microbench_kernel(float* __restrict__ out, int iters, unsigned long long* __restrict__ cycles) {
  __shared__ float4 sm[kMbThreads * 2];
  const int tid = threadIdx.x;
  float f[kMbUnroll];
  uint64_t d[kMbUnroll];
  uint32_t u[kMbUnroll];
#pragma unroll
  for (int i = 0; i < kMbUnroll; ++i) {
    f[i] = 1.0f + 1e-3f * (float)(tid + i);
    d[i] = pack2(f[i], -f[i]);
    u[i] = 0x9e3779b9u * (uint32_t)(tid + i + 1);
  }
  sm[tid] = make_float4(f[0], f[1], f[2], f[3]);
  sm[tid + kMbThreads] = make_float4(f[4], f[5], f[6], f[7]);
  const float k1 = 1.0000001f, k2 = 1e-7f;
  const uint64_t kk = pack2(k2, -k2), km = pack2(k1, k1);
  double g[kMbUnroll];
#pragma unroll
  for (int i = 0; i < kMbUnroll; ++i) g[i] = (double)f[i];
  const double gk1 = 1.0 + 1e-9 * (double)(tid & 3), gk2 = 1e-9;
  __syncthreads();
  const unsigned long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
    if constexpr (KIND == kMbFadd) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int i = 0; i < kMbUnroll; ++i) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(f[i]) : "f"(k2));
    } else if constexpr (KIND == kMbFfma) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int i = 0; i < kMbUnroll; ++i)
          asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[i]) : "f"(f[(i + 5) % kMbUnroll]), "f"(f[(i + 9) % kMbUnroll]));
    } else if constexpr (KIND == kMbFadd2) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int i = 0; i < kMbUnroll; ++i) asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(d[i]) : "l"(kk));
    } else if constexpr (KIND == kMbFfma2) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int i = 0; i < kMbUnroll; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(d[i]) : "l"(km), "l"(kk));
    } else if constexpr (KIND == kMbLop3) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int i = 0; i < kMbUnroll; ++i)
          asm volatile("lop3.b32 %0, %0, %1, 0x80000000, 0x6a;" : "+r"(u[i]) : "r"(u[(i + 3) % kMbUnroll]));
    } else if constexpr (KIND == kMbShf) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int i = 0; i < kMbUnroll; ++i)
          asm volatile("shf.l.wrap.b32 %0, %0, %1, 7;" : "+r"(u[i]) : "r"(u[(i + 3) % kMbUnroll]));
    } else if constexpr (KIND == kMbFadd2Lop3) {   // 1 FADD2 : 1 LOP3
#pragma unroll
      for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int i = 0; i < kMbUnroll; ++i) {
          asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(d[i]) : "l"(kk));
          asm volatile("lop3.b32 %0, %0, %1, 0x80000000, 0x6a;" : "+r"(u[i]) : "r"(u[(i + 3) % kMbUnroll]));
        }
    } else if constexpr (KIND == kMbFaddSign) {    // the round-1 chain: 7 FADD : 1 SHF : 1 LOP3
#pragma unroll
      for (int i = 0; i < kMbUnroll; ++i) {
#pragma unroll
        for (int r = 0; r < 7; ++r) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(f[(i + r) % kMbUnroll]) : "f"(k2));
        asm volatile("shf.l.wrap.b32 %0, %0, %1, 7;" : "+r"(u[i]) : "r"(u[(i + 3) % kMbUnroll]));
        asm volatile("lop3.b32 %0, %0, %1, 0x80000000, 0x6a;" : "+r"(u[(i + 1) % kMbUnroll]) : "r"(u[i]));
      }
    } else if constexpr (KIND == kMbFadd2Sign) {   // packed chain: 3 FADD2 + 1 FADD : 1 SHF : 1 LOP3 per element
#pragma unroll
      for (int i = 0; i < kMbUnroll; ++i) {
#pragma unroll
        for (int r = 0; r < 3; ++r) asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(d[(i + r) % kMbUnroll]) : "l"(kk));
        asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(f[i]) : "f"(k2));
        asm volatile("shf.l.wrap.b32 %0, %0, %1, 7;" : "+r"(u[i]) : "r"(u[(i + 3) % kMbUnroll]));
        asm volatile("lop3.b32 %0, %0, %1, 0x80000000, 0x6a;" : "+r"(u[(i + 1) % kMbUnroll]) : "r"(u[i]));
      }
    } else if constexpr (KIND == kMbFadd2Lop3Shf) {  // 2 FADD2 : 1 SHF : 1 LOP3
#pragma unroll
      for (int i = 0; i < kMbUnroll; ++i) {
#pragma unroll
        for (int r = 0; r < 2; ++r) asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(d[(i + r) % kMbUnroll]) : "l"(kk));
        asm volatile("shf.l.wrap.b32 %0, %0, %1, 7;" : "+r"(u[i]) : "r"(u[(i + 3) % kMbUnroll]));
        asm volatile("lop3.b32 %0, %0, %1, 0x80000000, 0x6a;" : "+r"(u[(i + 1) % kMbUnroll]) : "r"(u[i]));
      }
    } else if constexpr (KIND == kMbMufuCos) {
#pragma unroll
      for (int i = 0; i < kMbUnroll; ++i) asm volatile("cos.approx.ftz.f32 %0, %0;" : "+f"(f[i]));
    } else if constexpr (KIND == kMbLds128) {
#pragma unroll
      for (int i = 0; i < kMbUnroll; ++i) {
        float4 v;
        const uint32_t addr = (uint32_t)__cvta_generic_to_shared(&sm[(tid + 32 * i + it) & (2 * kMbThreads - 1)]);
        asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                     : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
        f[i] += v.x + v.w;
      }
    } else if constexpr (KIND == kMbShfl) {
#pragma unroll
      for (int i = 0; i < kMbUnroll; ++i) f[i] = __shfl_xor_sync(0xffffffffu, f[i], 1 + (i & 15));
    } else if constexpr (KIND == kMbDfma) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int i = 0; i < kMbUnroll; ++i)
          asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(g[i]) : "d"(gk1), "d"(gk2));
    } else if constexpr (KIND == kMbDmma) {          // 8 independent 8x8 accumulators (2 doubles per thread each)
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int i = 0; i < kMbUnroll; i += 2)
          asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                       : "+d"(g[i]), "+d"(g[i + 1]) : "d"(gk1), "d"(gk2));
    }
  }
  const unsigned long long t1 = clock64();
  float acc = 0.f;
#pragma unroll
  for (int i = 0; i < kMbUnroll; ++i) acc += f[i] + lo_of(d[i]) + __uint_as_float(u[i] & 0x3fffffffu) + (float)g[i];
  out[(size_t)blockIdx.x * kMbThreads + tid] = acc;
  if (tid == 0) cycles[blockIdx.x] = t1 - t0;
}

// lane-operations per thread and loop iteration (an f32x2 instruction counts two fp32 lane-operations)
static double mb_ops_per_iter(int kind) {
  switch (kind) {
    case kMbFadd: case kMbFfma: case kMbLop3: case kMbShf: return 4.0 * kMbUnroll;
    case kMbFadd2: case kMbFfma2: return 8.0 * kMbUnroll;
    case kMbFadd2Lop3: return 2.0 * kMbUnroll * 2;        // fp32 adds only
    case kMbFaddSign: return 7.0 * kMbUnroll;             // fp32 adds only
    case kMbFadd2Sign: return 7.0 * kMbUnroll;
    case kMbFadd2Lop3Shf: return 4.0 * kMbUnroll;
    case kMbMufuCos: case kMbShfl: return 1.0 * kMbUnroll;
    case kMbLds128: return 16.0 * kMbUnroll;              // bytes
    case kMbDfma: return 4.0 * kMbUnroll;                 // FP64 FMAs
    case kMbDmma: return 4.0 * (kMbUnroll / 2) * 8.0;     // FP64 FMAs: 8 x 8 x 4 = 256 per warp instruction, 8 per lane
    default: return 0.0;
  }
}

template <int K>
static int mb_launch(float* out, int iters, unsigned long long* cyc, int blocks, cudaStream_t st) {
  microbench_kernel<K><<<blocks, kMbThreads, 0, st>>>(out, iters, cyc);
  QMLL_LAUNCH_CHECK("microbench_kernel");
  return QMLL_OK;
}

int device_sm_count();

// ---- tcgen05.mma issue / operand timing: M = 128, kind::f16, both operands in shared memory, one CTA per SM; an elected
// lane issues `iters` x 4 x R MMAs of width N rotating over R accumulators, then commits and waits.  out[0] = clock64
// ticks of block 0 from the first issue to completion.
template <int N, int R>
__global__ void __launch_bounds__(128, 1) mma_clock_kernel(long long* out, int iters) {
  extern __shared__ uint8_t mb_smem_raw[];
  uint8_t* sm = reinterpret_cast<uint8_t*>(((uintptr_t)mb_smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ uint64_t bar;
  __shared__ uint32_t tptr;
  for (int i = threadIdx.x; i < (64 * 1024) / 4; i += 128) reinterpret_cast<uint32_t*>(sm)[i] = 0;
  if (threadIdx.x == 0) { mbar_init(&bar, 1); fence_mbarrier_init(); }
  if (threadIdx.x < 32) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&tptr)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  const uint32_t tb = tptr;
  if (threadIdx.x < 32) {
    const bool leader = elect_one_sync();
    const uint32_t tbu = __shfl_sync(0xffffffffu, tb, 0);
    const uint64_t a = make_kmajor_sw128_desc(smem_u32(sm)), b = make_kmajor_sw128_desc(smem_u32(sm + 16384));
    constexpr uint32_t idesc = (1u << 4) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    const long long t0 = clock64();
    if (leader) {
      for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int kk = 0; kk < 4; ++kk)
#pragma unroll
          for (int r = 0; r < R; ++r) umma<true>(tbu + r * N, a + 2 * kk, b + 2 * kk, idesc, 1u);
      }
      tcgen05_commit(&bar);
    }
    __syncwarp();
    mbar_wait(&bar, 0);
    const long long t1 = clock64();
    if (threadIdx.x == 0 && blockIdx.x == 0) out[0] = t1 - t0;
  }
  tcgen05_fence_before();
  __syncthreads();
  if (threadIdx.x < 32) {
    tcgen05_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tb) : "memory");
  }
}

template <int N, int R>
static int mma_clock_launch(long long* out, int iters, cudaStream_t st) {
  auto kern = mma_clock_kernel<N, R>;
  QMLL_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 70 * 1024));
  kern<<<device_sm_count(), 128, 70 * 1024, st>>>(out, iters);
  QMLL_LAUNCH_CHECK("mma_clock_kernel");
  return QMLL_OK;
}

}  // namespace qmll

using namespace qmll;

extern "C" int qmll_microbench_mma(int n, int accumulators, int iters, void* workspace, size_t workspace_bytes,
                                   void* cuda_stream) {
  if (iters < 1 || !workspace || workspace_bytes < 8) return QMLL_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  long long* out = static_cast<long long*>(workspace);
#define QMLL_MB(N_, R_) if (n == N_ && accumulators == R_) return mma_clock_launch<N_, R_>(out, iters, st);
  QMLL_MB(64, 1) QMLL_MB(64, 2) QMLL_MB(64, 4) QMLL_MB(96, 1) QMLL_MB(96, 2) QMLL_MB(96, 4)
  QMLL_MB(128, 1) QMLL_MB(128, 2) QMLL_MB(128, 4) QMLL_MB(256, 1) QMLL_MB(256, 2)
#undef QMLL_MB
  return QMLL_ERR_UNSUPPORTED;
}

extern "C" int qmll_microbench(int kind, int iters, int blocks_per_sm, void* workspace, size_t workspace_bytes,
                               double* ops_per_launch, int* n_blocks, void* cuda_stream) {
  if (kind < 0 || kind >= kMbCount || iters < 1 || blocks_per_sm < 1 || !ops_per_launch || !n_blocks)
    return QMLL_ERR_INVALID_ARG;
  const int blocks = device_sm_count() * blocks_per_sm;
  const size_t need = (size_t)blocks * kMbThreads * sizeof(float) + (size_t)blocks * sizeof(unsigned long long) + 512;
  if (!workspace || workspace_bytes < need) return QMLL_ERR_WORKSPACE;
  Carver ws(workspace, workspace_bytes);
  unsigned long long* cyc = ws.take<unsigned long long>(blocks);   // first: the caller reads cycles at offset 0
  float* out = ws.take<float>((size_t)blocks * kMbThreads);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  *ops_per_launch = mb_ops_per_iter(kind) * (double)iters * kMbThreads * blocks;
  *n_blocks = blocks;
  switch (kind) {
    case 0: return mb_launch<0>(out, iters, cyc, blocks, st);
    case 1: return mb_launch<1>(out, iters, cyc, blocks, st);
    case 2: return mb_launch<2>(out, iters, cyc, blocks, st);
    case 3: return mb_launch<3>(out, iters, cyc, blocks, st);
    case 4: return mb_launch<4>(out, iters, cyc, blocks, st);
    case 5: return mb_launch<5>(out, iters, cyc, blocks, st);
    case 6: return mb_launch<6>(out, iters, cyc, blocks, st);
    case 7: return mb_launch<7>(out, iters, cyc, blocks, st);
    case 8: return mb_launch<8>(out, iters, cyc, blocks, st);
    case 9: return mb_launch<9>(out, iters, cyc, blocks, st);
    case 10: return mb_launch<10>(out, iters, cyc, blocks, st);
    case 11: return mb_launch<11>(out, iters, cyc, blocks, st);
    case 12: return mb_launch<12>(out, iters, cyc, blocks, st);
    case 13: return mb_launch<13>(out, iters, cyc, blocks, st);
    case 14: return mb_launch<14>(out, iters, cyc, blocks, st);
    default: return QMLL_ERR_INVALID_ARG;
  }
}
