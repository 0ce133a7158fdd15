// ctr_measure_peaks (include/ctr.h): microbenchmarks of the on-chip units that bound the projector kernels,
// so that bench.py's roofline fractions rest on numbers measured on the device the bench runs on instead of
// datasheet products ("measure an FMA-issue microbenchmark on the box first").
// Not part of the reconstruction path. Every kernel is written with inline PTX so that the instruction
// counts used below are the ones that execute.
#include <cuda_runtime.h>

#include "../../include/ctr.h"

namespace {

constexpr int PK_THREADS = 256;
constexpr int PK_BLOCKS_PER_SM = 8;  // 2048 threads per SM: full occupancy

// 1. fp32 FMA: 8 independent chains per thread, 8 FFMA per loop trip and chain
__global__ void __launch_bounds__(PK_THREADS) k_peak_fma(int iters, float seed, float* sink) {
  float a0 = seed + threadIdx.x, a1 = a0 + 1.f, a2 = a0 + 2.f, a3 = a0 + 3.f, a4 = a0 + 4.f, a5 = a0 + 5.f, a6 = a0 + 6.f,
        a7 = a0 + 7.f;
  const float m = 0.999f, c = 0.001f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      asm volatile(
          "fma.rn.f32 %0, %0, %8, %9;\n\tfma.rn.f32 %1, %1, %8, %9;\n\tfma.rn.f32 %2, %2, %8, %9;\n\t"
          "fma.rn.f32 %3, %3, %8, %9;\n\tfma.rn.f32 %4, %4, %8, %9;\n\tfma.rn.f32 %5, %5, %8, %9;\n\t"
          "fma.rn.f32 %6, %6, %8, %9;\n\tfma.rn.f32 %7, %7, %8, %9;"
          : "+f"(a0), "+f"(a1), "+f"(a2), "+f"(a3), "+f"(a4), "+f"(a5), "+f"(a6), "+f"(a7)
          : "f"(m), "f"(c));
    }
  }
  const float s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
  if (s == 123.456f) sink[0] = s;
}

// 1b. packed fp32x2 FMA (FFMA2, sm_100): 8 independent 64-bit chains, 16 FMAs per instruction group
__global__ void __launch_bounds__(PK_THREADS) k_peak_fma2(int iters, float seed, float* sink) {
  unsigned long long a[8];
#pragma unroll
  for (int q = 0; q < 8; ++q) {
    const float lo = seed + threadIdx.x + q, hi = lo + 0.5f;
    asm volatile("mov.b64 %0, {%1, %2};" : "=l"(a[q]) : "f"(lo), "f"(hi));
  }
  unsigned long long m, c;
  asm volatile("mov.b64 %0, {%1, %1};" : "=l"(m) : "f"(0.999f));
  asm volatile("mov.b64 %0, {%1, %1};" : "=l"(c) : "f"(0.001f));
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      asm volatile(
          "fma.rn.f32x2 %0, %0, %8, %9;\n\tfma.rn.f32x2 %1, %1, %8, %9;\n\tfma.rn.f32x2 %2, %2, %8, %9;\n\t"
          "fma.rn.f32x2 %3, %3, %8, %9;\n\tfma.rn.f32x2 %4, %4, %8, %9;\n\tfma.rn.f32x2 %5, %5, %8, %9;\n\t"
          "fma.rn.f32x2 %6, %6, %8, %9;\n\tfma.rn.f32x2 %7, %7, %8, %9;"
          : "+l"(a[0]), "+l"(a[1]), "+l"(a[2]), "+l"(a[3]), "+l"(a[4]), "+l"(a[5]), "+l"(a[6]), "+l"(a[7])
          : "l"(m), "l"(c));
    }
  }
  unsigned long long s = 0;
#pragma unroll
  for (int q = 0; q < 8; ++q) s ^= a[q];
  if (s == 0x123456789abcdefull) sink[0] = 1.0f;
}

// 2. warp-instruction issue: FFMA (FMA pipe) and LOP3 / IADD3 (ALU pipe) interleaved, all independent:
// 8 FFMA + 8 integer instructions per group (a ring of data-dependent xor / add so that ptxas cannot fold them)
__global__ void __launch_bounds__(PK_THREADS) k_peak_issue(int iters, float seed, float* sink) {
  float a0 = seed + threadIdx.x, a1 = a0 + 1.f, a2 = a0 + 2.f, a3 = a0 + 3.f, a4 = a0 + 4.f, a5 = a0 + 5.f, a6 = a0 + 6.f,
        a7 = a0 + 7.f;
  unsigned b0 = threadIdx.x, b1 = b0 + 1, b2 = b0 + 2, b3 = b0 + 3, b4 = b0 + 4, b5 = b0 + 5, b6 = b0 + 6, b7 = b0 + 7;
  const float m = 0.999f, c = 0.001f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      asm volatile(
          "fma.rn.f32 %0, %0, %16, %17;\n\txor.b32 %8, %8, %9;\n\t"
          "fma.rn.f32 %1, %1, %16, %17;\n\tadd.u32 %9, %9, %10;\n\t"
          "fma.rn.f32 %2, %2, %16, %17;\n\txor.b32 %10, %10, %11;\n\t"
          "fma.rn.f32 %3, %3, %16, %17;\n\tadd.u32 %11, %11, %12;\n\t"
          "fma.rn.f32 %4, %4, %16, %17;\n\txor.b32 %12, %12, %13;\n\t"
          "fma.rn.f32 %5, %5, %16, %17;\n\tadd.u32 %13, %13, %14;\n\t"
          "fma.rn.f32 %6, %6, %16, %17;\n\txor.b32 %14, %14, %15;\n\t"
          "fma.rn.f32 %7, %7, %16, %17;\n\tadd.u32 %15, %15, %8;"
          : "+f"(a0), "+f"(a1), "+f"(a2), "+f"(a3), "+f"(a4), "+f"(a5), "+f"(a6), "+f"(a7), "+r"(b0), "+r"(b1), "+r"(b2),
            "+r"(b3), "+r"(b4), "+r"(b5), "+r"(b6), "+r"(b7)
          : "f"(m), "f"(c));
    }
  }
  const float s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
  const unsigned t = b0 ^ b1 ^ b2 ^ b3 ^ b4 ^ b5 ^ b6 ^ b7;
  if (s == 123.456f && t == 77u) sink[0] = s;
}

// 3. L1 data pipe, global loads that hit in L1: every thread reads 16 bytes (one LDG.E.128 = 4 wavefronts of
// 128 bytes per warp) from an 8 KB window of its block, addresses rotating so that nothing is hoisted
__global__ void __launch_bounds__(PK_THREADS) k_peak_l1(int iters, const float4* __restrict__ buf, float* sink) {
  const float4* base = buf + (size_t)blockIdx.x * 512;  // 512 float4 = 8 KB per block, 64 KB per SM at 8 blocks
  unsigned idx = threadIdx.x;
  float acc = 0.0f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      float4 v;
      asm volatile("ld.global.ca.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(base + (idx & 511u)));
      acc += (v.x + v.y) + (v.z + v.w);
      idx += 32u + (unsigned)u;
    }
  }
  if (acc == 123.456f) sink[0] = acc;
}

// 3b. L2 -> SM fabric: the same LDG.128 stream, but cache-global (ld.global.cg: not kept in L1) over a window of
// 2^21 float4 = 32 MiB that stays resident in the 126 MB L2; every warp reads 512 contiguous bytes (4 sectors
// of 4 lines) at a rotating, warp-dependent offset, like the 256-byte gathers of the projector kernels
__global__ void __launch_bounds__(PK_THREADS) k_peak_l2(int iters, const float4* __restrict__ buf, float* sink) {
  const unsigned lane = threadIdx.x & 31u;
  unsigned w = (blockIdx.x * (PK_THREADS / 32) + (threadIdx.x >> 5)) * 2654435761u;  // warp-dependent start chunk
  float acc = 0.0f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      float4 v;
      const float4* p = buf + ((size_t)(w & 0xffffu) * 32u + lane);  // chunk of 32 float4 out of 65536 chunks
      asm volatile("ld.global.cg.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
      acc += (v.x + v.y) + (v.z + v.w);
      w = w * 1664525u + 1013904223u;
    }
  }
  if (acc == 123.456f) sink[0] = acc;
}

// 4. shared memory: LDS.128 per thread (4 wavefronts per warp), conflict-free
__global__ void __launch_bounds__(PK_THREADS) k_peak_smem(int iters, float* sink) {
  __shared__ float4 sm[512];
  for (int t = threadIdx.x; t < 512; t += PK_THREADS) sm[t] = make_float4(t, 1.f, 2.f, 3.f);
  __syncthreads();
  unsigned idx = threadIdx.x;
  float acc = 0.0f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      float4 v;
      const unsigned addr = (unsigned)__cvta_generic_to_shared(&sm[idx & 511u]);
      asm volatile("ld.volatile.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
      acc += (v.x + v.y) + (v.z + v.w);
      idx += 32u;
    }
  }
  if (acc == 123.456f) sink[0] = acc;
}

// 5. HBM stream copy (read + write bytes), float4, grid-stride
__global__ void __launch_bounds__(PK_THREADS) k_peak_copy(const float4* __restrict__ src, float4* __restrict__ dst, size_t n) {
  for (size_t i = (size_t)blockIdx.x * PK_THREADS + threadIdx.x; i < n; i += (size_t)gridDim.x * PK_THREADS)
    dst[i] = __ldcs(src + i);
}

template <class F>
cudaError_t best_ms(F launch, int reps, float* best) {
  cudaEvent_t e0, e1;
  cudaError_t e = cudaEventCreate(&e0);
  if (e != cudaSuccess) return e;
  e = cudaEventCreate(&e1);
  if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
  *best = 1e30f;
  launch();  // warm-up
  for (int r = 0; r < reps && e == cudaSuccess; ++r) {
    cudaEventRecord(e0, 0);
    launch();
    cudaEventRecord(e1, 0);
    e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e == cudaSuccess && ms < *best) *best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (e == cudaSuccess) e = cudaGetLastError();
  return e;
}

}  // namespace

extern "C" int ctr_measure_peaks(ctr_peaks* out, int reps) {
  if (!out) return CTR_EINVAL;
  if (reps < 1) reps = 5;
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return CTR_ECUDA;
  if (prop.major != 10) return CTR_EARCH;
  const int sms = prop.multiProcessorCount, blocks = sms * PK_BLOCKS_PER_SM;
  const double threads = (double)blocks * PK_THREADS;
  const int iters = 2048;
  float* sink = nullptr;
  float4 *buf = nullptr, *src = nullptr, *dst = nullptr;
  const size_t ncopy = (size_t)1 << 26;  // 2^26 float4 = 1 GiB per array: far beyond the 126 MB L2
  cudaError_t e = cudaMalloc((void**)&sink, 256);
  if (e == cudaSuccess) e = cudaMalloc((void**)&buf, (size_t)blocks * 512 * sizeof(float4));
  if (e == cudaSuccess) e = cudaMalloc((void**)&src, ncopy * sizeof(float4));
  if (e == cudaSuccess) e = cudaMalloc((void**)&dst, ncopy * sizeof(float4));
  if (e == cudaSuccess) e = cudaMemset(buf, 0, (size_t)blocks * 512 * sizeof(float4));
  if (e == cudaSuccess) e = cudaMemset(src, 0, ncopy * sizeof(float4));
  float ms = 0.f;
  out->sm_count = sms;
  if (e == cudaSuccess) e = best_ms([&] { k_peak_fma<<<blocks, PK_THREADS>>>(iters, 1.0f, sink); }, reps, &ms);
  out->fma_tflops = threads * iters * 64.0 * 2.0 / (ms * 1e-3) / 1e12;
  out->issue_gwinst = threads / 32.0 * iters * 64.0 / (ms * 1e-3) / 1e9;
  if (e == cudaSuccess) e = best_ms([&] { k_peak_fma2<<<blocks, PK_THREADS>>>(iters, 1.0f, sink); }, reps, &ms);
  out->fma2_tflops = threads * iters * 64.0 * 4.0 / (ms * 1e-3) / 1e12;
  if (e == cudaSuccess) e = best_ms([&] { k_peak_issue<<<blocks, PK_THREADS>>>(iters, 1.0f, sink); }, reps, &ms);
  out->mixed_gwinst = threads / 32.0 * iters * 128.0 / (ms * 1e-3) / 1e9;
  if (e == cudaSuccess) e = best_ms([&] { k_peak_l1<<<blocks, PK_THREADS>>>(iters, buf, sink); }, reps, &ms);
  out->l1_tbs = threads * iters * 8.0 * 16.0 / (ms * 1e-3) / 1e12;
  if (e == cudaSuccess) e = best_ms([&] { k_peak_l2<<<blocks, PK_THREADS>>>(iters / 8, src, sink); }, reps, &ms);
  out->l2_tbs = threads * (iters / 8) * 8.0 * 16.0 / (ms * 1e-3) / 1e12;
  if (e == cudaSuccess) e = best_ms([&] { k_peak_smem<<<blocks, PK_THREADS>>>(iters, sink); }, reps, &ms);
  out->smem_tbs = threads * iters * 8.0 * 16.0 / (ms * 1e-3) / 1e12;
  if (e == cudaSuccess) e = best_ms([&] { k_peak_copy<<<sms * 16, PK_THREADS>>>(src, dst, ncopy); }, reps, &ms);
  out->hbm_copy_gbs = 2.0 * (double)ncopy * sizeof(float4) / (ms * 1e-3) / 1e9;
  if (sink) cudaFree(sink);
  if (buf) cudaFree(buf);
  if (src) cudaFree(src);
  if (dst) cudaFree(dst);
  if (e != cudaSuccess) { cudaGetLastError(); return e == cudaErrorMemoryAllocation ? CTR_ENOMEM : CTR_ECUDA; }
  return CTR_OK;
}
