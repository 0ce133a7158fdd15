// Shared device helpers of libctr (sm_100a). Nothing here is used by oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ctr {

// ---------------------------------------------------------------------------------------------
// V-wide "slice vectors". Internal arrays hold V = 1 (batch == 1) or V = 4 slices per element:
// element e of group g is at float offset (g * n + e) * V, i.e. a float4 when V = 4.
// ---------------------------------------------------------------------------------------------
template <int V> struct Pack;
template <> struct Pack<1> {
  __device__ static __forceinline__ void ld(const float* __restrict__ p, size_t e, float (&o)[1]) { o[0] = __ldg(p + e); }
  __device__ static __forceinline__ void ldcg(const float* p, size_t e, float (&o)[1]) { o[0] = __ldcg(p + e); }
  __device__ static __forceinline__ void st(float* p, size_t e, const float (&o)[1]) { p[e] = o[0]; }
};
template <> struct Pack<4> {
  __device__ static __forceinline__ void ld(const float* __restrict__ p, size_t e, float (&o)[4]) {
    float4 t = __ldg(reinterpret_cast<const float4*>(p) + e);
    o[0] = t.x; o[1] = t.y; o[2] = t.z; o[3] = t.w;
  }
  __device__ static __forceinline__ void ldcg(const float* p, size_t e, float (&o)[4]) {
    float4 t = __ldcg(reinterpret_cast<const float4*>(p) + e);
    o[0] = t.x; o[1] = t.y; o[2] = t.z; o[3] = t.w;
  }
  __device__ static __forceinline__ void st(float* p, size_t e, const float (&o)[4]) {
    reinterpret_cast<float4*>(p)[e] = make_float4(o[0], o[1], o[2], o[3]);
  }
};

// ---------------------------------------------------------------------------------------------
// Deterministic grid reduction: every block writes its partial sums, the block that arrives last
// (atomicInc ticket, self-resetting) adds all partials in a fixed order and calls fin(sums) from
// its thread 0. No floating-point atomics anywhere.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}

template <int N>
__device__ __forceinline__ void block_sum(double (&v)[N], double (*sm)[32], int tid, int nthreads) {
  const int lane = tid & 31, wid = tid >> 5, nw = (nthreads + 31) >> 5;
#pragma unroll
  for (int n = 0; n < N; ++n) {
    double w = warp_sum(v[n]);
    if (lane == 0) sm[n][wid] = w;
  }
  __syncthreads();
  if (wid == 0) {
#pragma unroll
    for (int n = 0; n < N; ++n) {
      double w = lane < nw ? sm[n][lane] : 0.0;
      v[n] = warp_sum(w);
    }
  }
  __syncthreads();
}

template <int N, class Fin>
__device__ __forceinline__ void grid_reduce(double (&v)[N], double* part, unsigned* counter, unsigned nblk,
                                            unsigned blk, int tid, int nthreads, Fin fin) {
  __shared__ double sm[N][32];
  __shared__ bool last;
  block_sum<N>(v, sm, tid, nthreads);
  if (tid == 0) {
#pragma unroll
    for (int n = 0; n < N; ++n) part[(size_t)blk * N + n] = v[n];
    __threadfence();
    unsigned t = atomicInc(counter, nblk - 1);
    last = (t == nblk - 1);
  }
  __syncthreads();
  if (!last) return;
  double acc[N];
#pragma unroll
  for (int n = 0; n < N; ++n) acc[n] = 0.0;
  for (unsigned b = tid; b < nblk; b += nthreads) {
#pragma unroll
    for (int n = 0; n < N; ++n) acc[n] += __ldcg(&part[(size_t)b * N + n]);
  }
  block_sum<N>(acc, sm, tid, nthreads);
  if (tid == 0) fin(acc);
}

// ---------------------------------------------------------------------------------------------
// Segmented variant for the slice-interleaved layout: thread tid holds N partial
// sums that belong to segment tid % LQ (LQ a power of two <= 16, block size NW * 32); the
// sums are kept apart per segment. Order of additions is fixed.
// ---------------------------------------------------------------------------------------------
template <int N, int NW>
__device__ __forceinline__ void block_sum_q(double (&v)[N], double (*sm)[NW][16], int LQ, int tid) {
  const int lane = tid & 31, wid = tid >> 5;
#pragma unroll
  for (int n = 0; n < N; ++n) {
    double w = v[n];
    for (int o = 16; o >= LQ; o >>= 1) w += __shfl_down_sync(0xffffffffu, w, o);
    if (lane < LQ) sm[n][wid][lane] = w;
  }
  __syncthreads();
  if (tid < LQ) {
#pragma unroll
    for (int n = 0; n < N; ++n) {
      double w = 0.0;
      for (int k = 0; k < NW; ++k) w += sm[n][k][tid];
      v[n] = w;
    }
  }
  __syncthreads();
}

// block partials of a segmented reduction: part[(blk * LQ + q) * N + n]; a finishing kernel
// (k_finish, ctr_api.cu) adds them over the blocks in a fixed order. A single finishing BLOCK inside the
// producing kernel cost 120-350 us per launch at 64 slices (measured in round 1): hence the extra tiny launch.
template <int N, int NW>
__device__ __forceinline__ void block_partials_q(double (&v)[N], int LQ, double* part, unsigned blk, int tid) {
  __shared__ double sm[N][NW][16];  // LQ <= 16
  block_sum_q<N, NW>(v, sm, LQ, tid);
  if (tid < LQ) {
#pragma unroll
    for (int n = 0; n < N; ++n) part[((size_t)blk * LQ + tid) * N + n] = v[n];
  }
}

// ---------------------------------------------------------------------------------------------
// The ONE definition of the system-matrix entry, used by both P (ctr_forward) and P^T (ctr_back).
//
// A ray is stored in grid-index coordinates with its driving axis d (the axis along which it
// advances fastest) and the other axis o:   o(dcoord) = x0 + m * dcoord,  |m| <= 1.
// Slab s of the driving axis spans dcoord in [s, s+1] (integers relative to the grid line c0).
// Within the slab the ray goes from oa = x0 + m*s to ob = x0 + m*(s+1) and therefore touches
// cells floor(oa) and floor(ob) of the other axis (equal, or adjacent because |m| <= 1).
// Its length inside the slab is L; the part in cell floor(oa) is |Xc - oa| * K with Xc the grid
// line between the two cells and K = L/|m|  (p_ij = intersection length).
// The floor is a fixed, branch-free round(o - 1/2) (ties may go either way; every use is consistent).
// ---------------------------------------------------------------------------------------------
#define CTR_MAGIC 12582912.0f      /* 1.5 * 2^23: adding it rounds to an integer held in the mantissa */
#define CTR_MAGIC_BITS 0x4B400000 /* bit pattern of CTR_MAGIC; bits(CTR_MAGIC + n) = CTR_MAGIC_BITS + n   */

struct SlabW {
  float ra, rb;  // CTR_MAGIC + cell index of the entry / exit cell (compare these, never recompute)
  float wa, wb;  // lengths (mm) in those cells; wb = 0 when ra == rb
};

// cell index (relative to the origin grid line) from a biased value
__device__ __forceinline__ int cell_of(float r) { return __float_as_int(r) - CTR_MAGIC_BITS; }
// biased value of an integer cell index (exact)
__device__ __forceinline__ float bias_of(int n) { return __int_as_float(CTR_MAGIC_BITS + n); }

__device__ __forceinline__ SlabW slab_weights(float oa, float ob, float L, float K) {
  SlabW w;
  w.ra = __fadd_rn(__fadd_rn(oa, -0.5f), CTR_MAGIC);  // "floor": round-to-nearest of oa - 1/2
  w.rb = __fadd_rn(__fadd_rn(ob, -0.5f), CTR_MAGIC);
  const bool same = (w.ra == w.rb);
  const float Xc = __fadd_rn(fmaxf(w.ra, w.rb), -CTR_MAGIC);  // grid line between the two cells
  const float w1 = fminf(__fmul_rn(fabsf(__fsub_rn(Xc, oa)), K), L);
  w.wa = same ? L : w1;
  w.wb = same ? 0.0f : __fsub_rn(L, w1);
  return w;
}

}  // namespace ctr
