// Stored system matrix in sliced-ELL form, for single problems (batch = 1: c1-c3, c5).
//
// PAPER.md:193 describes two strategies: trace the rays on the fly, or - "for small problems" that fit the
// GPU memory (4 GB on the paper's C1060) - precompute P and P^T as lookup tables. With 180 GB of HBM the
// second strategy covers every single-slice config (0.26 GB per matrix at 512^2 x 60 x 888) and even the 3D
// cone beam (c5: 4.4e9 non-zeros, ~40 GB per matrix). The tables hold exactly the values the on-the-fly
// kernels compute (the SAME visitor enumerates a row's entries in the SAME order in both), so the stored
// and the on-the-fly operators give identical bits and P^T remains the exact transpose of P.
//
// Layout: rows (rays for P, voxels for P^T) are taken 32 at a time (a warp); warp w owns cap[w] slabs of 32
// (index, weight) pairs at tab[off[w] + e * 32 + lane], cap[w] = the longest row of the warp, missing
// entries have weight 0. An application streams the table once with 256-byte coalesced reads.
#pragma once
#include <stdlib.h>

#include "ctr_common.cuh"
#include "ctr_internal.h"
#include "ctr_fan_geom.cuh"

namespace ctr {

// PASS 0: cap[w] = longest row of warp w;  PASS 1: fill. hits(row, visit) calls visit(index, weight) for
// every non-zero of the row, in the order the on-the-fly kernel adds them.
template <int PASS, class Hits>
__global__ void __launch_bounds__(128) k_ell_build(Dims d, Hits hits, size_t nrows, int* __restrict__ cap,
                                                   const size_t* __restrict__ off, float2* __restrict__ tab) {
  const size_t row = (size_t)blockIdx.x * 128 + threadIdx.x;
  const size_t warp = row >> 5;
  const int lane = threadIdx.x & 31;
  if ((warp << 5) >= nrows) return;  // whole warp
  int n = 0;
  if (PASS == 0) {
    if (row < nrows) hits(d, row, [&](int, float) { ++n; });
    const int m = __reduce_max_sync(0xffffffffu, n);
    if (lane == 0) cap[warp] = m;
  } else {
    float2* slab = tab + off[warp] + lane;
    if (row < nrows)
      hits(d, row, [&](int idx, float wt) {
        slab[(size_t)n * 32] = make_float2(__int_as_float(idx), wt);
        ++n;
      });
    const int m = cap[warp];
    for (int e = n; e < m; ++e) slab[(size_t)e * 32] = make_float2(0.0f, 0.0f);
  }
}

// out[row] = sum_e w_e in[idx_e]  (+ the CGLS epilogues of the on-the-fly kernels, V = 1)
//   ROLE 0 (P):   MODE 0 plain, MODE 1 out = bs - P x, MODE 2 also delta = ||out||^2 -> a = gamma/delta
//   ROLE 1 (P^T): MODE 0 plain, MODE 2 also u += a s for the voxel
// SPLIT > 1 (P of a single 2D slice): a ray's entries are dealt round-robin to SPLIT consecutive table rows
// (threads) and the partial sums are added by a fixed shuffle tree - a slice has too few rays to hide the
// latency of ~n dependent gathers per ray otherwise.
template <int SPLIT, class Hits>
struct SplitHits {
  Hits hits;
  template <class Visit>
  __device__ __forceinline__ void operator()(const Dims& d, size_t row, Visit visit) const {
    const int part = (int)(row % SPLIT);
    int e = 0;
    hits(d, row / SPLIT, [&](int idx, float wt) {
      if (e % SPLIT == part) visit(idx, wt);
      ++e;
    });
  }
};

template <int ROLE, int MODE, int SPLIT>
__global__ void __launch_bounds__(128) k_ell_apply(size_t nrows, const int* __restrict__ cap, const size_t* __restrict__ off,
                                                   const float2* __restrict__ tab, const float* __restrict__ in,
                                                   float* __restrict__ out, const float* __restrict__ aux,
                                                   float* __restrict__ u_img, Scal sc, double* part, unsigned* counter) {
  const size_t row = (size_t)blockIdx.x * 128 + threadIdx.x;
  const size_t warp = row >> 5;
  float acc = 0.0f;
  if ((warp << 5) < nrows) {
    const int m = __ldg(&cap[warp]);
    const float2* slab = tab + __ldg(&off[warp]) + (threadIdx.x & 31);
#pragma unroll 4
    for (int e = 0; e < m; ++e) {
      const float2 h = __ldcs(slab + (size_t)e * 32);
      if (h.y != 0.0f) acc = fmaf(h.y, __ldg(in + __float_as_int(h.x)), acc);
    }
  }
  if (SPLIT > 1) {
#pragma unroll
    for (int o = 1; o < SPLIT; o <<= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  }
  if (row < nrows && row % SPLIT == 0) {
    const size_t orow = row / SPLIT;
    if (ROLE == 0 && MODE == 1) acc = __ldg(aux + orow) - acc;
    out[orow] = acc;
    if (ROLE == 1 && MODE == 2) u_img[orow] = fmaf(sc.a[0], __ldcg(aux + orow), __ldcg(u_img + orow));
  } else {
    acc = 0.0f;
  }
  if (ROLE == 0 && MODE == 2) {
    double v[1] = {(double)acc * (double)acc};
    if (counter) {
      // few blocks (a 2D slice): the block that arrives last adds the partials and forms a = gamma/delta here
      grid_reduce<1>(v, part, counter, gridDim.x, blockIdx.x, threadIdx.x, 128, [&](double(&sum)[1]) {
        const double gamma = sc.gamma[0];
        sc.a[0] = (sum[0] > 0.0 && gamma > 0.0) ? (float)(gamma / sum[0]) : 0.0f;  // S4
      });
    } else {
      // many blocks (c5: 92 000, where that single finishing block took ~0.6 ms): block partials only, k_finish
      // adds them with 1024 threads
      __shared__ double sm[1][32];
      block_sum<1>(v, sm, threadIdx.x, 128);
      if (threadIdx.x == 0) part[blockIdx.x] = v[0];
    }
  }
}

// Build a table for `nrows` rows. Best effort: leaves t.tab == nullptr (the caller then uses the on-the-fly
// kernel) when the table does not fit in free device memory or ctr_geometry.flags has CTR_GEOM_NO_TABLES.
template <class Hits>
static int ell_build(ctr_handle* h, Hits hits, size_t nrows, EllTable& t) {
  t.tab = nullptr; t.cap = nullptr; t.off = nullptr; t.nrows = nrows;
  if (h->g.flags & CTR_GEOM_NO_TABLES) return CTR_OK;
  const size_t nwarp = (nrows + 31) / 32;
  const unsigned nblk = (unsigned)((nrows + 127) / 128);
  if (cudaMalloc((void**)&t.cap, sizeof(int) * nwarp) != cudaSuccess) { cudaGetLastError(); t.cap = nullptr; return CTR_OK; }
  k_ell_build<0, Hits><<<nblk, 128>>>(h->d, hits, nrows, t.cap, nullptr, nullptr);
  CTR_LAUNCHED(h);
  int* cap = (int*)malloc(sizeof(int) * nwarp);
  size_t* off = (size_t*)malloc(sizeof(size_t) * nwarp);
  if (!cap || !off) { free(cap); free(off); return CTR_ENOMEM; }
  CTR_CUDA(h, cudaMemcpy(cap, t.cap, sizeof(int) * nwarp, cudaMemcpyDeviceToHost));
  size_t total = 0;
  for (size_t w = 0; w < nwarp; ++w) { off[w] = total; total += (size_t)cap[w] * 32; }
  free(cap);
  size_t free_b = 0, total_b = 0;
  cudaMemGetInfo(&free_b, &total_b);
  const size_t need = total * sizeof(float2) + nwarp * sizeof(size_t);
  bool ok = total > 0 && need + ((size_t)4 << 30) < free_b;  // leave 4 GiB of head room
  if (ok && cudaMalloc((void**)&t.off, sizeof(size_t) * nwarp) != cudaSuccess) { cudaGetLastError(); t.off = nullptr; ok = false; }
  if (ok && cudaMalloc((void**)&t.tab, total * sizeof(float2)) != cudaSuccess) { cudaGetLastError(); t.tab = nullptr; ok = false; }
  if (!ok) {
    free(off);
    if (t.off) cudaFree(t.off);
    cudaFree(t.cap);
    t.tab = nullptr; t.cap = nullptr; t.off = nullptr;
    return CTR_OK;
  }
  cudaError_t ce = cudaMemcpy(t.off, off, sizeof(size_t) * nwarp, cudaMemcpyHostToDevice);
  free(off);
  if (ce != cudaSuccess) return cuda_fail(h, ce, "ell_build: offsets");
  k_ell_build<1, Hits><<<nblk, 128>>>(h->d, hits, nrows, t.cap, t.off, t.tab);
  CTR_LAUNCHED(h);
  CTR_CUDA(h, cudaDeviceSynchronize());
  t.bytes = need;
  return CTR_OK;
}

#ifndef ELL_BLOCKED
#define ELL_BLOCKED 1
#endif
// vol[z][y][x] -> blocked copy (blk_index, ctr_fan_geom.cuh); one thread per element of the blocked array
static __global__ void __launch_bounds__(256) k_to_blocked(int nx, int ny, int nz, const float* __restrict__ vol, float* __restrict__ out) {
  const size_t o = (size_t)blockIdx.x * 256 + threadIdx.x;
  if (o >= (size_t)nx * ny * nz) return;
  const int xi = (int)(o & 7), yi = (int)((o >> 3) & 3);
  size_t t = o >> 5;
  const int tx = (int)(t % (nx >> 3));
  t /= (nx >> 3);
  const int ty = (int)(t % (ny >> 2)), z = (int)(t / (ny >> 2));
  out[o] = __ldg(vol + ((size_t)z * ny + (ty << 2) + yi) * nx + (tx << 3) + xi);
}

template <int SPLIT>
static int ell_forward(ctr_handle* h, const EllTable& t, const float* img, float* out, int mode, const float* bs,
                       cudaStream_t st) {
  const unsigned nblk = (unsigned)((t.nrows + 127) / 128);
  unsigned* cnt = h->counters;
  if (mode == 0) k_ell_apply<0, 0, SPLIT><<<nblk, 128, 0, st>>>(t.nrows, t.cap, t.off, t.tab, img, out, bs, nullptr, h->sc, h->part, cnt);
  else if (mode == 1) k_ell_apply<0, 1, SPLIT><<<nblk, 128, 0, st>>>(t.nrows, t.cap, t.off, t.tab, img, out, bs, nullptr, h->sc, h->part, cnt);
  else k_ell_apply<0, 2, SPLIT><<<nblk, 128, 0, st>>>(t.nrows, t.cap, t.off, t.tab, img, out, bs, nullptr, h->sc, h->part,
                                                      nblk > 8192 ? nullptr : cnt);
  CTR_LAUNCHED(h);
  if (mode == 2 && nblk > 8192) return reduce_finish(h, CTR_FIN_ALPHA, 1, (int)nblk, 0, 0, 0, st);  // a = gamma/||P s||^2
  return CTR_OK;
}

static int ell_back(ctr_handle* h, const EllTable& t, const float* sino, float* out, int mode, const float* s, float* u,
                    cudaStream_t st) {
  const unsigned nblk = (unsigned)((t.nrows + 127) / 128);
  if (mode == 0) k_ell_apply<1, 0, 1><<<nblk, 128, 0, st>>>(t.nrows, t.cap, t.off, t.tab, sino, out, s, u, h->sc, h->part, h->counters);
  else k_ell_apply<1, 2, 1><<<nblk, 128, 0, st>>>(t.nrows, t.cap, t.off, t.tab, sino, out, s, u, h->sc, h->part, h->counters);
  CTR_LAUNCHED(h);
  return CTR_OK;
}

}  // namespace ctr
