// 2D fan-beam projector pair for BATCHED slices (batch > 1) on sm_100a, slice-interleaved layout.
//
// Layout "SI": element e (pixel or ray) of super-group gs holds the LQ*4 slices of
// that super-group contiguously: float4 index (gs * n + e) * LQ + q, lane c of quad q = slice
// (gs * LQ + q) * 4 + c. With 64 slices (LQ = 16) one pixel is 256 contiguous bytes.
//
// A sub-warp of LQ lanes owns one ray (P) or one pixel (P^T); lane q of the sub-warp carries quad q of
// the slices. The geometry of a ray/pixel is therefore evaluated ONCE for all slices, in parallel over
// the lanes of the sub-warp (lane q evaluates slab sb+q of the ray, or view k0+q of the pixel), and the
// results are handed round by shuffles / a shared-memory queue. Every image or sinogram access of a
// sub-warp is one contiguous LQ*16-byte segment: the L1 wavefront count per useful byte, which bound
// the one-thread-per-ray kernel (profiles/r1a_ncu_full_c4.md: 7.5 wavefronts per LDG.128), drops to the
// minimum of one wavefront per 128 bytes.
//
// Both kernels evaluate the SAME slab_weights() on the SAME fp32 ray table as the single-slice kernels
// of ctr_fan.cu, so every p_ij is identical bit for bit in P and P^T (exact transpose up to summation
// order).   P: PAPER.md:87-89 (Eq. 1), :193.   P^T: PAPER.md:193, :471 (A3'); north_star.
#include <limits.h>
#include <stdlib.h>

#include "ctr_common.cuh"
#include "ctr_internal.h"
#include "ctr_fan_geom.cuh"

namespace ctr {

#define FULL 0xffffffffu

__device__ __forceinline__ void fma4(float (&acc)[4], float w, const float4 f) {
  acc[0] = fmaf(w, f.x, acc[0]);
  acc[1] = fmaf(w, f.y, acc[1]);
  acc[2] = fmaf(w, f.z, acc[2]);
  acc[3] = fmaf(w, f.w, acc[3]);
}

// The 4 x 4 outer product acc[p][c] += w_p y_c of the quad gather with packed fp32x2 instructions (FFMA2, sm_100):
// A[pp][0] = (acc[2pp][0], acc[2pp+1][1]), A[pp][1] = (acc[2pp][1], acc[2pp+1][0]), A[pp][2] = (acc[2pp][2],
// acc[2pp+1][3]), A[pp][3] = (acc[2pp][3], acc[2pp+1][2]): the weight pairs (w0,w1), (w2,w3) and the slice pairs
// (y0,y1), (y2,y3) are the register pairs the 128-bit loads deliver, the swapped slice pairs cost two moves:
// 8 FFMA2 + moves instead of 16 FFMA per table entry, the same fma per accumulator in the same order (same bits).
__device__ __forceinline__ void outer16(float2 (&A)[2][4], const float4 w, const float4 y) {
  const float2 w01 = make_float2(w.x, w.y), w23 = make_float2(w.z, w.w);
  const float2 y01 = make_float2(y.x, y.y), y10 = make_float2(y.y, y.x);
  const float2 y23 = make_float2(y.z, y.w), y32 = make_float2(y.w, y.z);
  A[0][0] = __ffma2_rn(w01, y01, A[0][0]);
  A[0][1] = __ffma2_rn(w01, y10, A[0][1]);
  A[0][2] = __ffma2_rn(w01, y23, A[0][2]);
  A[0][3] = __ffma2_rn(w01, y32, A[0][3]);
  A[1][0] = __ffma2_rn(w23, y01, A[1][0]);
  A[1][1] = __ffma2_rn(w23, y10, A[1][1]);
  A[1][2] = __ffma2_rn(w23, y23, A[1][2]);
  A[1][3] = __ffma2_rn(w23, y32, A[1][3]);
}
#ifndef SI_BACK_FMA2
#define SI_BACK_FMA2 1
#endif

// ------------------------------------------------------------------------------------------------
// a1  P. Sub-warp per ray. The slab loop runs over a warp-uniform range in batches of LQ slabs: lane q
// evaluates slab_weights() of slab sb+q (closed form per slab, no dependence between slabs), then the
// sub-warp walks the LQ slabs in ascending order, every lane accumulating its own quad of slices.
// MODE 0: out = P x    MODE 1: out = bs - P x (CGLS r0)
// MODE 2: out = P x and delta = ||out||^2 per slice -> a = gamma/delta (App. I step 1, :423)
// ------------------------------------------------------------------------------------------------
#ifndef SI_FWD_MINB
#define SI_FWD_MINB 4 /* 64 registers: more loads in flight than the 40 ptxas picks unprompted (6.76 vs 7.07 ms per step) */
#endif
// (A ray-quad table for P, the mirror image of the quad gather below, was built and measured in round 1:
// 7.2-7.5 ms per step against 6.75 ms for this kernel - adjacent rays share pixels along one axis only.)
#ifndef SI_FWD_WARPS
#define SI_FWD_WARPS 8 /* warps per block (16 adjacent rays at LQ = 16); 4, 16 and 32 measured slower */
#endif

// H = float4 slice quads per lane: a sub-warp has SW = LQ / H lanes. With 64 slices (LQ = 16) H = 2: a ray is
// carried by 8 lanes that read the pixel as two contiguous 128-byte halves (quads l and l + 8), so a warp holds
// four rays and one broadcast record read serves twice as many FMAs. ncu (round 1, H = 1) had the L1 data pipe
// as the busiest unit at 78 %, a third of its wavefronts being the record traffic through shared memory; the
// global wavefronts are already the algorithmic minimum (one per 128 bytes gathered).
template <int LQ, int H, int MODE>
__global__ void __launch_bounds__(SI_FWD_WARPS * 32, SI_FWD_MINB) k_si_forward(Dims d, const float4* __restrict__ rays,
                                                    const float4* __restrict__ img, float4* __restrict__ out,
                                                    const float4* __restrict__ bs, Scal sc, double* part,
                                                    unsigned* counter) {
  constexpr int SW = LQ / H;   // lanes per ray
  constexpr int RW = 32 / SW;  // rays per warp
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int q = lane % SW, sub = lane / SW;
  const int r = (blockIdx.x * SI_FWD_WARPS + warp) * RW + sub;
  const int gs = blockIdx.y;
  const bool live = r < d.nray;
  float acc[H][4];
#pragma unroll
  for (int hh = 0; hh < H; ++hh)
#pragma unroll
    for (int c = 0; c < 4; ++c) acc[hh][c] = 0.0f;
  // per-slab records {pa, wa, pb, wb} of the sub-warp's ray, written by the lane that evaluated the slab
  // and read back as one broadcast LDS.128 per slab (a shuffle costs an L1 data-pipe wavefront each; four
  // of them per slab were 40 % of the pipe, measured in round 1). Rows are padded by one entry so that the
  // sub-warps of a warp hit different banks. (Interleaving the two rays' records per slab, and 8-byte
  // records with the second length recomputed as L - wa, were measured: no gain / 50 % slower.)
  __shared__ float4 slab[SI_FWD_WARPS][RW][SW + 1];
  float4* myslab = slab[warp][sub];

  float x0 = 0.0f, m = 0.0f, L = 0.0f, K = 0.0f;
  bool xdrv = false;
  int s0 = INT_MAX, s1 = 0;
  if (live) {
    const float4 R = __ldg(&rays[r]);
    x0 = R.x; m = R.y; L = fabsf(R.z); K = R.w;
    xdrv = R.z < 0.0f;
  }
  const int n_drv = xdrv ? d.nx : d.ny, n_oth = xdrv ? d.ny : d.nx;
  const int c_drv = xdrv ? d.c0x : d.c0y, c_oth = xdrv ? d.c0y : d.c0x;
  if (live) {
    // slabs in which the ray can be inside [-c_oth, n_oth - c_oth) (same margins as k_fan_forward)
    s0 = 0; s1 = n_drv;
    const float lo = (float)(-c_oth) - 1.0f, hi = (float)(n_oth - c_oth) + 1.0f;
    if (m != 0.0f) {
      float t1 = (lo - x0) / m, t2 = (hi - x0) / m;
      float tmin = fminf(t1, t2), tmax = fmaxf(t1, t2);
      tmin = fminf(fmaxf(tmin, -1.0e6f), 1.0e6f);
      tmax = fminf(fmaxf(tmax, -1.0e6f), 1.0e6f);
      s0 = max(0, (int)floorf(tmin) + c_drv - 2);
      s1 = min(n_drv, (int)ceilf(tmax) + c_drv + 2);
    } else if (x0 < lo || x0 > hi) {
      s1 = 0;
    }
    if (s1 <= s0) { s0 = INT_MAX; s1 = 0; }
  }
  const int w_lo = __reduce_min_sync(FULL, s0), w_hi = __reduce_max_sync(FULL, s1);
  const float4* base = img + (size_t)gs * d.npix * LQ + q;
  asm volatile("" : "+l"(base));  // keep the pointer in a register pair: one IMAD.WIDE per address
  const int st_drv = (xdrv ? 1 : d.nx) * LQ;  // float4 stride of one slab step
  const int st_oth = (xdrv ? d.nx : 1) * LQ;  // float4 stride of one cell of the other axis

  for (int sb = w_lo; sb < w_hi; sb += SW) {
    const int s = sb + q;
    int pa = 0, pb = 0;
    float wa = 0.0f, wb = 0.0f;
    if (s >= s0 && s < s1) {
      const float y = (float)(s - c_drv);
      const float oa = fmaf(m, y, x0), ob = fmaf(m, y + 1.0f, x0);
      const SlabW w = slab_weights(oa, ob, L, K);
      const int ia = cell_of(w.ra) + c_oth, ib = cell_of(w.rb) + c_oth;
      const bool va = (unsigned)ia < (unsigned)n_oth;
      const bool vb = w.wb != 0.0f && (unsigned)ib < (unsigned)n_oth;
      if (va) {
        pa = s * st_drv + ia * st_oth;
        wa = w.wa;
        if (vb) { pb = s * st_drv + ib * st_oth; wb = w.wb; }
      } else if (vb) {
        pa = s * st_drv + ib * st_oth;
        wa = w.wb;
      }
    }
    __syncwarp();
    myslab[q] = make_float4(__int_as_float(pa), wa, __int_as_float(pb), wb);
    __syncwarp();
#pragma unroll
    for (int t = 0; t < SW; ++t) {
      const float4 rec = myslab[t];
      if (rec.y != 0.0f) {
        const float4* pa4 = base + __float_as_int(rec.x);
#pragma unroll
        for (int hh = 0; hh < H; ++hh) fma4(acc[hh], rec.y, __ldg(pa4 + hh * SW));
      }
      if (rec.w != 0.0f) {
        const float4* pb4 = base + __float_as_int(rec.z);
#pragma unroll
        for (int hh = 0; hh < H; ++hh) fma4(acc[hh], rec.w, __ldg(pb4 + hh * SW));
      }
    }
  }
  if (live) {
#pragma unroll
    for (int hh = 0; hh < H; ++hh) {
      const size_t e = ((size_t)gs * d.nray + r) * LQ + q + hh * SW;
      if (MODE == 1) {
        const float4 b = __ldg(bs + e);
        acc[hh][0] = b.x - acc[hh][0]; acc[hh][1] = b.y - acc[hh][1]; acc[hh][2] = b.z - acc[hh][2]; acc[hh][3] = b.w - acc[hh][3];
      }
      out[e] = make_float4(acc[hh][0], acc[hh][1], acc[hh][2], acc[hh][3]);
    }
  }
  if (MODE == 2) {
    // ||out||^2 per slice: the thread's 4 H sums belong to slice quads q + hh SW
    double v[4 * H];
#pragma unroll
    for (int hh = 0; hh < H; ++hh)
#pragma unroll
      for (int c = 0; c < 4; ++c) v[hh * 4 + c] = live ? (double)acc[hh][c] * (double)acc[hh][c] : 0.0;
    __shared__ double sm[4 * H][SI_FWD_WARPS][16];
    block_sum_q<4 * H, SI_FWD_WARPS>(v, sm, SW, threadIdx.x);
    if (threadIdx.x < SW) {
      double* dst = part + ((size_t)gs * gridDim.x + blockIdx.x) * LQ * 4;
#pragma unroll
      for (int hh = 0; hh < H; ++hh)
#pragma unroll
        for (int c = 0; c < 4; ++c) dst[(threadIdx.x + hh * SW) * 4 + c] = v[hh * 4 + c];
    }
  }
}

// ------------------------------------------------------------------------------------------------
// a1 with the stored matrix (NEXT-2; "pre-calculate the projection matrix and save it ... as a lookup
// table", CGLS by sparse matrix products): P as ONE table shared by all slices - per ray its non-zeros
// (pixel index * LQ, p_ij) in the order k_si_forward adds them, padded to whole chunks of 16 - applied to the
// 64 slices at once, i.e. a sparse-matrix x dense-matrix product with the slices as columns. 8 B x nnz(P) =
// 236 MB at 512^2 / 60 x 888 streamed from HBM per application, against 64 x nnz x 4 B gathered through the L1s.
// The sub-warp of a ray loads a chunk of 16 entries with one coalesced 128-byte read, hands them round through
// shared memory two at a time (one LDS.128 = two entries) and every lane does one 16-byte gather and 4 FMAs per
// entry: no slab arithmetic, no empty slabs, no divergent second-cell branch. Same p_ij bits (the table is
// filled by the row visitor the on-the-fly kernels share), same order of additions per ray: identical results.
// ------------------------------------------------------------------------------------------------
template <int PASS>
__global__ void __launch_bounds__(128) k_raytab_build(Dims d, const float4* __restrict__ rays, int* __restrict__ cnt,
                                                      const unsigned* __restrict__ off, float2* __restrict__ tab, int scale) {
  const int r = blockIdx.x * 128 + threadIdx.x;
  if (r >= d.nray) return;
  FanRayHits hits{rays};
  int n = 0;
  if (PASS == 0) {
    hits(d, (size_t)r, [&](int, float) { ++n; });
    cnt[r] = n;
  } else {
    float2* dst = tab + off[r];
    hits(d, (size_t)r, [&](int idx, float wt) { dst[n++] = make_float2(__int_as_float(idx * scale), wt); });
    const int padded = (cnt[r] + 15) / 16 * 16;
    for (; n < padded; ++n) dst[n] = make_float2(0.0f, 0.0f);
  }
}

#ifndef SI_TAB_MINB
#define SI_TAB_MINB SI_FWD_MINB
#endif
template <int LQ, int MODE>
__global__ void __launch_bounds__(SI_FWD_WARPS * 32, SI_TAB_MINB) k_si_forward_tab(Dims d, const int* __restrict__ cnt,
                                                    const unsigned* __restrict__ off, const float2* __restrict__ tab,
                                                    const float4* __restrict__ img, float4* __restrict__ out,
                                                    const float4* __restrict__ bs, Scal sc, double* part) {
  constexpr int RW = 32 / LQ;  // rays per warp
  constexpr int CH = 16;       // entries per chunk and ray (a 128-byte line of the table)
  static_assert(LQ <= CH && CH % LQ == 0, "chunk must be a whole number of sub-warp loads");
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int q = lane % LQ, sub = lane / LQ;
  const int r = (blockIdx.x * SI_FWD_WARPS + warp) * RW + sub;
  const int gs = blockIdx.y;
  const bool live = r < d.nray;
  __shared__ __align__(16) float2 ent[SI_FWD_WARPS][RW][CH + 2];  // rows padded: sub-warps in different banks
  float2* mine = ent[warp][sub];
  float acc[4] = {0.0f, 0.0f, 0.0f, 0.0f};
  const int n = live ? __ldg(&cnt[r]) : 0;
  const int nmax = __reduce_max_sync(FULL, n);
  const float2* src = tab + (live ? __ldg(&off[r]) : 0u);
  const float4* base = img + (size_t)gs * d.npix * LQ + q;
  asm volatile("" : "+l"(base));
  for (int e0 = 0; e0 < nmax; e0 += CH) {
    __syncwarp();
#pragma unroll
    for (int c = 0; c < CH / LQ; ++c) {
      const int e = e0 + c * LQ + q;
      mine[c * LQ + q] = e < n ? __ldcs(src + e) : make_float2(0.0f, 0.0f);  // streamed once per application
    }
    __syncwarp();
#pragma unroll
    for (int t = 0; t < CH; t += 2) {
      const float4 two = *reinterpret_cast<const float4*>(mine + t);  // entries t and t + 1
      if (two.y != 0.0f) fma4(acc, two.y, __ldg(base + __float_as_int(two.x)));
      if (two.w != 0.0f) fma4(acc, two.w, __ldg(base + __float_as_int(two.z)));
    }
  }
  if (live) {
    const size_t e = ((size_t)gs * d.nray + r) * LQ + q;
    if (MODE == 1) {
      const float4 b = __ldg(bs + e);
      acc[0] = b.x - acc[0]; acc[1] = b.y - acc[1]; acc[2] = b.z - acc[2]; acc[3] = b.w - acc[3];
    }
    out[e] = make_float4(acc[0], acc[1], acc[2], acc[3]);
  }
  if (MODE == 2) {
    double v[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) v[c] = live ? (double)acc[c] * (double)acc[c] : 0.0;
    block_partials_q<4, SI_FWD_WARPS>(v, LQ, part + (size_t)gs * gridDim.x * LQ * 4, blockIdx.x, threadIdx.x);
  }
}

// built once per handle (ctr_create), best effort: without it k_si_forward computes the entries on the fly
int si_build_raytab(ctr_handle* h) {
  const Dims& d = h->d;
  h->rt_tab = nullptr; h->rt_cnt = nullptr; h->rt_off = nullptr; h->rt_bytes = 0;
  if (h->g.flags & (CTR_GEOM_NO_TABLES | CTR_GEOM_NO_STORED_P)) return CTR_OK;
  if ((size_t)d.npix * d.LQ >= (1u << 31)) return CTR_OK;
  if (cudaMalloc((void**)&h->rt_cnt, sizeof(int) * (size_t)d.nray) != cudaSuccess) { cudaGetLastError(); h->rt_cnt = nullptr; return CTR_OK; }
  const unsigned nblk = (unsigned)((d.nray + 127) / 128);
  k_raytab_build<0><<<nblk, 128>>>(d, h->rays, h->rt_cnt, nullptr, nullptr, d.LQ);
  CTR_LAUNCHED(h);
  int* cnt = (int*)malloc(sizeof(int) * (size_t)d.nray);
  unsigned* off = (unsigned*)malloc(sizeof(unsigned) * (size_t)d.nray);
  if (!cnt || !off) { free(cnt); free(off); return CTR_ENOMEM; }
  CTR_CUDA(h, cudaMemcpy(cnt, h->rt_cnt, sizeof(int) * (size_t)d.nray, cudaMemcpyDeviceToHost));
  unsigned long long total = 0;
  for (int r = 0; r < d.nray; ++r) { off[r] = (unsigned)total; total += (unsigned long long)(cnt[r] + 15) / 16 * 16; }
  free(cnt);
  bool ok = total > 0 && total < (1ull << 32);
  if (ok && cudaMalloc((void**)&h->rt_off, sizeof(unsigned) * (size_t)d.nray) != cudaSuccess) { cudaGetLastError(); h->rt_off = nullptr; ok = false; }
  if (ok && cudaMalloc((void**)&h->rt_tab, sizeof(float2) * total) != cudaSuccess) { cudaGetLastError(); h->rt_tab = nullptr; ok = false; }
  if (!ok) {
    free(off);
    if (h->rt_off) cudaFree(h->rt_off);
    cudaFree(h->rt_cnt);
    h->rt_tab = nullptr; h->rt_cnt = nullptr; h->rt_off = nullptr;
    return CTR_OK;
  }
  cudaError_t ce = cudaMemcpy(h->rt_off, off, sizeof(unsigned) * (size_t)d.nray, cudaMemcpyHostToDevice);
  free(off);
  if (ce != cudaSuccess) return cuda_fail(h, ce, "si_build_raytab: offsets");
  k_raytab_build<1><<<nblk, 128>>>(d, h->rays, h->rt_cnt, h->rt_off, h->rt_tab, d.LQ);
  CTR_LAUNCHED(h);
  CTR_CUDA(h, cudaDeviceSynchronize());
  h->rt_bytes = sizeof(float2) * total;
  return CTR_OK;
}

// ------------------------------------------------------------------------------------------------
// a2  P^T (gather). Sub-warp per pixel; a block is a TX x TY tile of pixels, so the sinogram segments
// it reads overlap in L1. Views are taken LQ at a time: lane q looks up the bins of view k0+q whose
// rays cross the pixel (window table win2, or fan_window() when the table is not usable) and evaluates
// their weights; non-zero (ray, weight) pairs are compacted into a per-pixel shared-memory queue in a
// fixed order (candidate slot, then view), which the sub-warp then drains: one contiguous LQ*16-byte
// sinogram read and 4 FMAs per lane per pair. No atomics; the order of additions is fixed.
// MODE 0: out = P^T y     MODE 2: out = g = P^T r and, fused, u += a s (App. I step 2)
// ------------------------------------------------------------------------------------------------
#define SI_CH 4 /* candidate slots per lane between two drains of the queue */

template <int LQ, int MODE, int TABLE>
__global__ void __launch_bounds__(256) k_si_back(Dims d, const float4* __restrict__ rays,
                                                 const float2* __restrict__ views,
                                                 const unsigned short* __restrict__ win2,
                                                 const float4* __restrict__ sino, float4* __restrict__ out,
                                                 const float4* __restrict__ s_img, float4* __restrict__ u_img, Scal sc) {
  constexpr int PB = 256 / LQ;  // pixels per block
  constexpr int TX = PB >= 64 ? 8 : 4, TY = PB / TX;
  __shared__ float2 queue[PB][LQ * SI_CH];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int q = lane % LQ, sub = lane / LQ;
  const int pl = warp * (32 / LQ) + sub;
  const int i = blockIdx.x * TX + pl % TX, j = blockIdx.y * TY + pl / TX;
  const int gs = blockIdx.z;
  const bool live = i < d.nx && j < d.ny;
  float acc[4] = {0.0f, 0.0f, 0.0f, 0.0f};
  const float fi = (float)(i - d.c0x), fj = (float)(j - d.c0y);
  const float bi = bias_of(i - d.c0x), bj = bias_of(j - d.c0y);
  const float px = fmaf((float)i + 0.5f, d.dx, d.xlo), py = fmaf((float)j + 0.5f, d.dy, d.ylo);
  const int pix = j * d.nx + i;
  const unsigned submask = (LQ == 32 ? FULL : ((1u << LQ) - 1u)) << (sub * LQ);
  const unsigned lt = submask & ((1u << lane) - 1u);
  const float4* sg = sino + (size_t)gs * d.nray * LQ + q;
  float2* myq = queue[pl];

  for (int k0 = 0; k0 < d.nviews; k0 += LQ) {
    const int k = k0 + q;
    int b_lo = 0, cnt = 0;
    if (live && k < d.nviews) {
      if (TABLE) {
        const unsigned w = __ldg(&win2[(size_t)pix * d.nvp + k]);
        b_lo = (int)(w >> 4);
        cnt = (int)(w & 15u);
      } else {
        int b_hi;
        fan_window(d, __ldg(&views[k]), px, py, b_lo, b_hi);
        cnt = max(0, b_hi - b_lo + 1);
      }
    }
    const int maxc = __reduce_max_sync(FULL, cnt);
    for (int c0 = 0; c0 < maxc; c0 += SI_CH) {
      int n = 0;
#pragma unroll
      for (int c = 0; c < SI_CH; ++c) {
        float wt = 0.0f;
        int idx = 0;
        if (c0 + c < cnt) {
          idx = k * d.nu + b_lo + c0 + c;
          wt = fan_pixel_weight(__ldg(&rays[idx]), fi, fj, bi, bj);
        }
        const bool hit = wt != 0.0f;
        const unsigned bal = __ballot_sync(FULL, hit) & submask;
        if (hit) myq[n + __popc(bal & lt)] = make_float2(__int_as_float(idx), wt);
        n += __popc(bal);
      }
      __syncwarp();
#pragma unroll 4
      for (int e = 0; e < n; ++e) {
        const float2 h = myq[e];
        fma4(acc, h.y, __ldg(sg + (size_t)__float_as_int(h.x) * LQ));
      }
      __syncwarp();
    }
  }
  if (!live) return;
  const size_t e = ((size_t)gs * d.npix + pix) * LQ + q;
  out[e] = make_float4(acc[0], acc[1], acc[2], acc[3]);
  if (MODE == 2) {
    const float4 sv = __ldcg(s_img + e);
    float4 uv = __ldcg(u_img + e);
    const int sl = (gs * LQ + q) * 4;
    uv.x = fmaf(sc.a[sl + 0], sv.x, uv.x);
    uv.y = fmaf(sc.a[sl + 1], sv.y, uv.y);
    uv.z = fmaf(sc.a[sl + 2], sv.z, uv.z);
    uv.w = fmaf(sc.a[sl + 3], sv.w, uv.w);
    u_img[e] = uv;
  }
}

// ------------------------------------------------------------------------------------------------
// a2 with the quad hit table ("store P^T as a lookup table" - the strategy the paper uses
// when the matrix fits; here ~380 MB at 512^2 x 60 x 888, shared by all slices, against 180 GB of HBM).
// A sub-warp owns a 2 x 2 quad of pixels: neighbouring pixels are crossed by largely the same rays, so one
// 256-byte sinogram read serves up to four pixels (x 4 slices per lane = 16 FMAs): ~250 reads per quad
// instead of 4 x 113, which is what the L1 data pipe - the bound of this kernel - sees.
// qidx[quad][e] = ray index * LQ (or -1: padding), qwts[quad][e] = p_ij of that ray in pixels
// (i0,j0), (i0+1,j0), (i0,j0+1), (i0+1,j0+1); views ascending, bins ascending. The weights are the values
// fan_pixel_weight() returns (0 where the ray misses the pixel), so P^T stays the bit-exact transpose of P
// and every pixel adds its non-zero terms in the same order as the single-slice kernel (a ray that misses a
// pixel of the quad adds 0 * y: the inputs must be finite, include/ctr.h).
// (A 2 x 4 tile was measured too: 6.3 ms per step against 4.2 ms - 32 accumulators per lane cost more in
// occupancy than the extra sharing saves.)
// ------------------------------------------------------------------------------------------------
template <int TABLE>
__global__ void __launch_bounds__(128) k_qhits_build(Dims d, const float4* __restrict__ rays,
                                                     const float2* __restrict__ views,
                                                     const unsigned short* __restrict__ win, int* __restrict__ qcnt,
                                                     int* __restrict__ qidx, float4* __restrict__ qwts, int HC,
                                                     int scale) {
  const int nqx = (d.nx + 1) / 2, nqy = (d.ny + 1) / 2;
  const int qx = blockIdx.x * 32 + threadIdx.x, qy = blockIdx.y * 4 + threadIdx.y;
  if (qx >= nqx || qy >= nqy) return;
  const int quad = qy * nqx + qx;
  float fi[4], fj[4], bi[4], bj[4], px[4], py[4];
  int pix[4];
  bool ok[4];
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    const int i = 2 * qx + (p & 1), j = 2 * qy + (p >> 1);
    ok[p] = i < d.nx && j < d.ny;
    fi[p] = (float)(i - d.c0x); fj[p] = (float)(j - d.c0y);
    bi[p] = bias_of(i - d.c0x); bj[p] = bias_of(j - d.c0y);
    px[p] = fmaf((float)i + 0.5f, d.dx, d.xlo); py[p] = fmaf((float)j + 0.5f, d.dy, d.ylo);
    pix[p] = j * d.nx + i;
  }
  int n = 0;
  for (int k = 0; k < d.nviews; ++k) {
    int lo[4], hi[4], b_lo = INT_MAX, b_hi = -1;
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      lo[p] = 0; hi[p] = -1;
      if (!ok[p]) continue;
      if (TABLE) {
        const unsigned w = __ldg(&win[(size_t)k * d.npix + pix[p]]);
        lo[p] = (int)(w >> 4);
        hi[p] = lo[p] + (int)(w & 15u) - 1;
      } else {
        fan_window(d, __ldg(&views[k]), px[p], py[p], lo[p], hi[p]);
      }
      if (hi[p] >= lo[p]) { b_lo = min(b_lo, lo[p]); b_hi = max(b_hi, hi[p]); }
    }
    for (int b = b_lo; b <= b_hi; ++b) {
      const float4 R = __ldg(&rays[k * d.nu + b]);
      float w[4];
      bool any = false;
#pragma unroll
      for (int p = 0; p < 4; ++p) {
        w[p] = (b >= lo[p] && b <= hi[p]) ? fan_pixel_weight(R, fi[p], fj[p], bi[p], bj[p]) : 0.0f;
        any |= w[p] != 0.0f;
      }
      if (any) {
        if (qidx) {
          qidx[(size_t)quad * HC + n] = (k * d.nu + b) * scale;
          qwts[(size_t)quad * HC + n] = make_float4(w[0], w[1], w[2], w[3]);
        }
        ++n;
      }
    }
  }
  if (qidx) {
    for (int e = n; e < HC; ++e) {
      qidx[(size_t)quad * HC + e] = -1;
      qwts[(size_t)quad * HC + e] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    }
  } else {
    qcnt[quad] = n;
  }
}

#ifndef SI_BACK_MINB
#define SI_BACK_MINB 4
#endif
template <int LQ, int MODE>
__global__ void __launch_bounds__(256, SI_BACK_MINB) k_si_back_quad(Dims d, const int* __restrict__ qcnt,
                                                      const int* __restrict__ qidx, const float4* __restrict__ qwts,
                                                      int HC, const float4* __restrict__ sino, float4* __restrict__ out,
                                                      const float4* __restrict__ s_img, float4* __restrict__ u_img,
                                                      Scal sc) {
  constexpr int PB = 256 / LQ;  // quads per block
  constexpr int TX = PB >= 64 ? 8 : 4, TY = PB / TX;
  // chunk of LQ table entries per quad, handed round through shared memory (broadcast reads; rows padded
  // so that the sub-warps of a warp use different banks)
  __shared__ float4 chw[PB][LQ + 1];
  __shared__ __align__(16) int chi[PB][LQ + 4];  // rows 16-byte aligned: four indices per LDS.128
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int q = lane % LQ, sub = lane / LQ;
  const int pl = warp * (32 / LQ) + sub;
  const int nqx = (d.nx + 1) / 2, nqy = (d.ny + 1) / 2;
  const int qx = blockIdx.x * TX + pl % TX, qy = blockIdx.y * TY + pl / TX;
  const int gs = blockIdx.z;
  const bool live = qx < nqx && qy < nqy;
  const int quad = live ? qy * nqx + qx : 0;
  float acc[4][4];
#pragma unroll
  for (int p = 0; p < 4; ++p)
#pragma unroll
    for (int c = 0; c < 4; ++c) acc[p][c] = 0.0f;
  float2 A2[2][4];
#pragma unroll
  for (int pp = 0; pp < 2; ++pp)
#pragma unroll
    for (int c = 0; c < 4; ++c) A2[pp][c] = make_float2(0.0f, 0.0f);
  const int cnt = live ? __ldg(&qcnt[quad]) : 0;
  const int wmax = __reduce_max_sync(FULL, cnt);
  const float4* sg = sino + (size_t)gs * d.nray * LQ + q;
  asm volatile("" : "+l"(sg));
  const int* ip = qidx + (size_t)quad * HC + q;
  const float4* wp = qwts + (size_t)quad * HC + q;
  for (int e0 = 0; e0 < wmax; e0 += LQ) {
    int id = -1;
    float4 w4 = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    if (e0 + q < cnt) { id = __ldcs(ip + e0); w4 = __ldcs(wp + e0); }  // streamed once per application
    __syncwarp();
    chi[pl][q] = id;
    chw[pl][q] = w4;
    __syncwarp();
    if (LQ % 4 == 0) {
      // the ray indices four at a time: a broadcast LDS.128 per four entries instead of an LDS.32 per entry (shared
      // memory and the gathers share the L1 data pipe, which bounds this kernel)
#pragma unroll
      for (int t4 = 0; t4 < LQ / 4; ++t4) {
        const int4 i4 = *reinterpret_cast<const int4*>(&chi[pl][4 * t4]);
        const int its[4] = {i4.x, i4.y, i4.z, i4.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          if (its[k] >= 0) {
            const float4 w = chw[pl][4 * t4 + k];
            const float4 y = __ldg(sg + its[k]);
            if (SI_BACK_FMA2) {
              outer16(A2, w, y);
            } else {
              fma4(acc[0], w.x, y);
              fma4(acc[1], w.y, y);
              fma4(acc[2], w.z, y);
              fma4(acc[3], w.w, y);
            }
          }
        }
      }
    } else {
#pragma unroll
      for (int t = 0; t < LQ; ++t) {
        const int it = chi[pl][t];
        if (it >= 0) {
          const float4 w = chw[pl][t];
          const float4 y = __ldg(sg + it);
          fma4(acc[0], w.x, y);
          fma4(acc[1], w.y, y);
          fma4(acc[2], w.z, y);
          fma4(acc[3], w.w, y);
        }
      }
    }
  }
  if (!live) return;
  if (SI_BACK_FMA2 && LQ % 4 == 0) {
#pragma unroll
    for (int pp = 0; pp < 2; ++pp) {
      acc[2 * pp][0] = A2[pp][0].x; acc[2 * pp][1] = A2[pp][1].x; acc[2 * pp][2] = A2[pp][2].x; acc[2 * pp][3] = A2[pp][3].x;
      acc[2 * pp + 1][0] = A2[pp][1].y; acc[2 * pp + 1][1] = A2[pp][0].y; acc[2 * pp + 1][2] = A2[pp][3].y; acc[2 * pp + 1][3] = A2[pp][2].y;
    }
  }
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    const int i = 2 * qx + (p & 1), j = 2 * qy + (p >> 1);
    if (i >= d.nx || j >= d.ny) continue;
    const size_t e = ((size_t)gs * d.npix + (size_t)j * d.nx + i) * LQ + q;
    out[e] = make_float4(acc[p][0], acc[p][1], acc[p][2], acc[p][3]);
    if (MODE == 2) {
      const float4 sv = __ldcg(s_img + e);
      float4 uv = __ldcg(u_img + e);
      const int sl = (gs * LQ + q) * 4;
      uv.x = fmaf(sc.a[sl + 0], sv.x, uv.x);
      uv.y = fmaf(sc.a[sl + 1], sv.y, uv.y);
      uv.z = fmaf(sc.a[sl + 2], sv.z, uv.z);
      uv.w = fmaf(sc.a[sl + 3], sv.w, uv.w);
      u_img[e] = uv;
    }
  }
}

// built once per handle (ctr_create); on allocation failure the on-the-fly kernel k_si_back is used
int si_build_hits(ctr_handle* h) {
  const Dims& d = h->d;
  h->qidx = nullptr;
  h->qwts = nullptr;
  h->hits_cap = 0;
  if (h->g.flags & CTR_GEOM_NO_TABLES) return CTR_OK;
  const int nqx = (d.nx + 1) / 2, nqy = (d.ny + 1) / 2, nquad = nqx * nqy;
  if (cudaMalloc((void**)&h->qcnt, sizeof(int) * (size_t)nquad) != cudaSuccess) { cudaGetLastError(); h->qcnt = nullptr; return CTR_OK; }
  dim3 grid((nqx + 31) / 32, (nqy + 3) / 4), block(32, 4);
  if (h->win_ok) k_qhits_build<1><<<grid, block>>>(d, h->rays, h->views, h->win, h->qcnt, nullptr, nullptr, 0, d.LQ);
  else k_qhits_build<0><<<grid, block>>>(d, h->rays, h->views, h->win, h->qcnt, nullptr, nullptr, 0, d.LQ);
  CTR_LAUNCHED(h);
  // capacity = largest count, rounded up to a whole number of 16-entry chunks
  int* host = (int*)malloc(sizeof(int) * (size_t)nquad);
  if (!host) return CTR_ENOMEM;
  CTR_CUDA(h, cudaMemcpy(host, h->qcnt, sizeof(int) * (size_t)nquad, cudaMemcpyDeviceToHost));
  int mx = 0;
  for (int p = 0; p < nquad; ++p) mx = host[p] > mx ? host[p] : mx;
  free(host);
  const int HC = (mx + 15) / 16 * 16;
  if (HC == 0 || (size_t)d.nray * d.LQ >= (1u << 31)) return CTR_OK;
  if (cudaMalloc((void**)&h->qidx, sizeof(int) * (size_t)nquad * HC) != cudaSuccess) { cudaGetLastError(); h->qidx = nullptr; return CTR_OK; }
  if (cudaMalloc((void**)&h->qwts, sizeof(float4) * (size_t)nquad * HC) != cudaSuccess) {
    cudaGetLastError();
    cudaFree(h->qidx);
    h->qidx = nullptr; h->qwts = nullptr;
    return CTR_OK;
  }
  h->hits_cap = HC;
  if (h->win_ok) k_qhits_build<1><<<grid, block>>>(d, h->rays, h->views, h->win, h->qcnt, h->qidx, h->qwts, HC, d.LQ);
  else k_qhits_build<0><<<grid, block>>>(d, h->rays, h->views, h->win, h->qcnt, h->qidx, h->qwts, HC, d.LQ);
  CTR_LAUNCHED(h);
  CTR_CUDA(h, cudaDeviceSynchronize());
  return CTR_OK;
}

// ------------------------------------------------------------------------------------------------
// Layout conversions. ABI: [B][n] floats. Planar (TV kernels): [G][n] float4. SI: [GS][n][LQ] float4.
// Slice (g, c) of the planar layout is slice (gs * LQ + q, c) of SI with g = gs * LQ + q.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_si_from_abi(const float* __restrict__ src, float4* __restrict__ dst, int n,
                                                     int B, int LQ) {
  const int e = blockIdx.x * 256 + threadIdx.x, g = blockIdx.y;
  if (e >= n) return;
  float o[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const int sl = 4 * g + c;
    o[c] = sl < B ? __ldg(src + (size_t)sl * n + e) : 0.0f;
  }
  dst[((size_t)(g / LQ) * n + e) * LQ + g % LQ] = make_float4(o[0], o[1], o[2], o[3]);
}

__global__ void __launch_bounds__(256) k_si_to_abi(const float4* __restrict__ src, float* __restrict__ dst, int n,
                                                   int B, int LQ) {
  const int e = blockIdx.x * 256 + threadIdx.x, g = blockIdx.y;
  if (e >= n) return;
  const float4 t = __ldg(src + ((size_t)(g / LQ) * n + e) * LQ + g % LQ);
  const float o[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const int sl = 4 * g + c;
    if (sl < B) dst[(size_t)sl * n + e] = o[c];
  }
}

// planar <-> SI through a shared-memory tile of 32 elements x LQ quads (both sides coalesced)
template <int TO_SI>
__global__ void __launch_bounds__(256) k_si_planar(const float4* __restrict__ src, float4* __restrict__ dst, int n,
                                                   int LQ) {
  __shared__ float4 tile[16][33];  // LQ <= 16
  const int gs = blockIdx.y, e0 = blockIdx.x * 32, tid = threadIdx.x;
  const int nel = 32 * LQ;
  if (TO_SI) {
    for (int t = tid; t < nel; t += 256) {
      const int qq = t >> 5, el = t & 31;
      if (e0 + el < n) tile[qq][el] = __ldcg(src + ((size_t)(gs * LQ + qq) * n + e0 + el));
    }
    __syncthreads();
    for (int t = tid; t < nel; t += 256) {
      const int el = t / LQ, qq = t % LQ;
      if (e0 + el < n) dst[((size_t)gs * n + e0 + el) * LQ + qq] = tile[qq][el];
    }
  } else {
    for (int t = tid; t < nel; t += 256) {
      const int el = t / LQ, qq = t % LQ;
      if (e0 + el < n) tile[qq][el] = __ldcg(src + ((size_t)gs * n + e0 + el) * LQ + qq);
    }
    __syncthreads();
    for (int t = tid; t < nel; t += 256) {
      const int qq = t >> 5, el = t & 31;
      if (e0 + el < n) dst[(size_t)(gs * LQ + qq) * n + e0 + el] = tile[qq][el];
    }
  }
}

int si_from_abi(ctr_handle* h, const float* src, float* dst, size_t n, cudaStream_t st) {
  dim3 grid((unsigned)((n + 255) / 256), h->d.G);
  ProfScope prof(h, CTR_PROF_LAYOUT, st);
  k_si_from_abi<<<grid, 256, 0, st>>>(src, (float4*)dst, (int)n, h->d.B, h->d.LQ);
  CTR_LAUNCHED(h);
  return CTR_OK;
}
int si_to_abi(ctr_handle* h, const float* src, float* dst, size_t n, cudaStream_t st) {
  dim3 grid((unsigned)((n + 255) / 256), h->d.G);
  ProfScope prof(h, CTR_PROF_LAYOUT, st);
  k_si_to_abi<<<grid, 256, 0, st>>>((const float4*)src, dst, (int)n, h->d.B, h->d.LQ);
  CTR_LAUNCHED(h);
  return CTR_OK;
}
int si_from_planar(ctr_handle* h, const float* src, float* dst, size_t n, cudaStream_t st) {
  dim3 grid((unsigned)((n + 31) / 32), h->d.GS);
  ProfScope prof(h, CTR_PROF_LAYOUT, st);
  k_si_planar<1><<<grid, 256, 0, st>>>((const float4*)src, (float4*)dst, (int)n, h->d.LQ);
  CTR_LAUNCHED(h);
  return CTR_OK;
}
int si_to_planar(ctr_handle* h, const float* src, float* dst, size_t n, cudaStream_t st) {
  dim3 grid((unsigned)((n + 31) / 32), h->d.GS);
  ProfScope prof(h, CTR_PROF_LAYOUT, st);
  k_si_planar<0><<<grid, 256, 0, st>>>((const float4*)src, (float4*)dst, (int)n, h->d.LQ);
  CTR_LAUNCHED(h);
  return CTR_OK;
}

// ------------------------------------------------------------------------------------------------
// host side: dispatch on LQ (1, 2, 4, 8, 16)
// ------------------------------------------------------------------------------------------------
#ifndef SI_FWD_H
#define SI_FWD_H 1 /* float4 slice quads per lane of k_si_forward at LQ = 16 (1: a ray per 16 lanes, 2: per 8 lanes) */
#endif
template <int LQ>
static int si_forward_t(ctr_handle* h, const float* img, float* out, int mode, const float* bs, cudaStream_t st) {
  const Dims& d = h->d;
  constexpr int H = LQ == 16 ? SI_FWD_H : 1;
  const int rays_per_block = SI_FWD_WARPS * (32 / (LQ / H)), nt = SI_FWD_WARPS * 32;
  dim3 grid((d.nray + rays_per_block - 1) / rays_per_block, d.GS);
  unsigned* cnt = h->counters + 0 * d.G;
  const float4 *im = (const float4*)img, *b4 = (const float4*)bs;
  float4* o4 = (float4*)out;
  ProfScope prof(h, CTR_PROF_FORWARD, st);
  if (h->rt_tab) {
    dim3 tgrid((d.nray + SI_FWD_WARPS * (32 / LQ) - 1) / (SI_FWD_WARPS * (32 / LQ)), d.GS);
    if (mode == 0) k_si_forward_tab<LQ, 0><<<tgrid, nt, 0, st>>>(d, h->rt_cnt, h->rt_off, h->rt_tab, im, o4, b4, h->sc, h->part);
    else if (mode == 1) k_si_forward_tab<LQ, 1><<<tgrid, nt, 0, st>>>(d, h->rt_cnt, h->rt_off, h->rt_tab, im, o4, b4, h->sc, h->part);
    else k_si_forward_tab<LQ, 2><<<tgrid, nt, 0, st>>>(d, h->rt_cnt, h->rt_off, h->rt_tab, im, o4, b4, h->sc, h->part);
    CTR_LAUNCHED(h);
    if (mode == 2) return reduce_finish(h, CTR_FIN_ALPHA, 4, (int)tgrid.x, 0, 0, 0, st);
    return CTR_OK;
  }
  if (mode == 0) k_si_forward<LQ, H, 0><<<grid, nt, 0, st>>>(d, h->rays, im, o4, b4, h->sc, h->part, cnt);
  else if (mode == 1) k_si_forward<LQ, H, 1><<<grid, nt, 0, st>>>(d, h->rays, im, o4, b4, h->sc, h->part, cnt);
  else k_si_forward<LQ, H, 2><<<grid, nt, 0, st>>>(d, h->rays, im, o4, b4, h->sc, h->part, cnt);
  CTR_LAUNCHED(h);
  if (mode == 2) return reduce_finish(h, CTR_FIN_ALPHA, 4, (int)grid.x, 0, 0, 0, st);  // a = gamma/||P s||^2
  return CTR_OK;
}

template <int LQ>
static int si_back_t(ctr_handle* h, const float* sino, float* out, int mode, const float* s, float* u, cudaStream_t st) {
  const Dims& d = h->d;
  constexpr int PB = 256 / LQ, TX = PB >= 64 ? 8 : 4, TY = PB / TX;
  dim3 grid((d.nx + TX - 1) / TX, (d.ny + TY - 1) / TY, d.GS);
  const float4 *y4 = (const float4*)sino, *s4 = (const float4*)s;
  float4 *o4 = (float4*)out, *u4 = (float4*)u;
  ProfScope prof(h, CTR_PROF_BACK, st);
  if (h->qwts) {
    dim3 qgrid(((d.nx + 1) / 2 + TX - 1) / TX, ((d.ny + 1) / 2 + TY - 1) / TY, d.GS);
    if (mode == 0) k_si_back_quad<LQ, 0><<<qgrid, 256, 0, st>>>(d, h->qcnt, h->qidx, h->qwts, h->hits_cap, y4, o4, s4, u4, h->sc);
    else k_si_back_quad<LQ, 2><<<qgrid, 256, 0, st>>>(d, h->qcnt, h->qidx, h->qwts, h->hits_cap, y4, o4, s4, u4, h->sc);
    CTR_LAUNCHED(h);
    return CTR_OK;
  }
#define CTR_SI_BACK(M, T) k_si_back<LQ, M, T><<<grid, 256, 0, st>>>(d, h->rays, h->views, h->win2, y4, o4, s4, u4, h->sc)
  if (h->win_ok) {
    if (mode == 0) CTR_SI_BACK(0, 1); else CTR_SI_BACK(2, 1);
  } else {
    if (mode == 0) CTR_SI_BACK(0, 0); else CTR_SI_BACK(2, 0);
  }
#undef CTR_SI_BACK
  CTR_LAUNCHED(h);
  return CTR_OK;
}

int si_forward(ctr_handle* h, const float* img, float* out, int mode, const float* bs, cudaStream_t st) {
  switch (h->d.LQ) {
    case 1: return si_forward_t<1>(h, img, out, mode, bs, st);
    case 2: return si_forward_t<2>(h, img, out, mode, bs, st);
    case 4: return si_forward_t<4>(h, img, out, mode, bs, st);
    case 8: return si_forward_t<8>(h, img, out, mode, bs, st);
    default: return si_forward_t<16>(h, img, out, mode, bs, st);
  }
}

int si_back(ctr_handle* h, const float* sino, float* out, int mode, const float* s, float* u, cudaStream_t st) {
  switch (h->d.LQ) {
    case 1: return si_back_t<1>(h, sino, out, mode, s, u, st);
    case 2: return si_back_t<2>(h, sino, out, mode, s, u, st);
    case 4: return si_back_t<4>(h, sino, out, mode, s, u, st);
    case 8: return si_back_t<8>(h, sino, out, mode, s, u, st);
    default: return si_back_t<16>(h, sino, out, mode, s, u, st);
  }
}

}  // namespace ctr
