// Edge-preserving TV step for sm_100a (2D slices with V = 1 or 4 slices per element, and 3D volumes
// with V = 1): face magnitudes A3, exact sigma order statistic, weights, gradient A2, Armijo trials and
// the descent update (+ positivity clamp).
//   A3 / weights : PAPER.md:106-110 (Eq. 4-5, sigma from the histogram), :458-463
//   A2 / gradient: PAPER.md:151-153 (Eq. 9-10), :453
//   Armijo       : PAPER.md:149;  clamp: PAPER.md:157, :173
// Readings: S5/S7/S8 faces, S9/S10 sigma = exact q-quantile, S11 eps, S12 replicate border
// with zero border flux, S14 Armijo constants, S22 3D generalisation.
#include <limits.h>

#include "ctr_common.cuh"
#include "ctr_internal.h"

namespace ctr {

#ifndef TV_GMINB
#define TV_GMINB 5 /* min blocks per SM of k_tv_gradient (register budget) */
#endif
#ifndef TV_FMINB
#define TV_FMINB 6 /* same for k_tv_faces */
#endif


// ---------------------------------------------------------------------------------------------
// Neighbourhood access. The stencil of A2/A3 around voxel p needs f at p + {-1,0,1}^ndim minus
// the far corners; we load the full 3x3 (2D) or 3x3x3 (3D) window with per-axis clamped indices
// (replicate border, S12) so the formulas below need no special cases. The loads go through L1 (ld.global.nc):
// neighbouring threads share eight of the nine cells, and with cache-bypassing loads every one of them went to
// L2 (round 1: k_tv_faces at 0 % L1 hits and 19 % of DRAM peak). The image is never written by a kernel that
// reads it through a window.
// ---------------------------------------------------------------------------------------------
template <int V, int ND>
struct Window {
  float c[ND == 3 ? 3 : 1][3][3][V];  // [dz+1][dy+1][dx+1][slice]
};

template <int V, int ND>
__device__ __forceinline__ void load_window(const Dims& d, const float* __restrict__ f, int g, int i, int j, int k,
                                            Window<V, ND>& w) {
  const float* base = f + (size_t)g * d.npix * V;
  int xi[3] = {max(i - 1, 0), i, min(i + 1, d.nx - 1)};
  int yj[3] = {max(j - 1, 0), j, min(j + 1, d.ny - 1)};
  if (ND == 3) {
    int zk[3] = {max(k - 1, 0), k, min(k + 1, d.nz - 1)};
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b)
#pragma unroll
        for (int c = 0; c < 3; ++c)
          Pack<V>::ld(base, ((size_t)zk[a] * d.ny + yj[b]) * d.nx + xi[c], w.c[ND == 3 ? a : 0][b][c]);
  } else {
#pragma unroll
    for (int b = 0; b < 3; ++b)
#pragma unroll
      for (int c = 0; c < 3; ++c) Pack<V>::ld(base, (size_t)yj[b] * d.nx + xi[c], w.c[0][b][c]);
  }
}

// N0^2 of the face between window cell q and q + e_A (A3), for slice lane s.
// q is given as window coordinates (qz,qy,qx) in {0,1,2}; the caller guarantees q+e_A and q +- e_T
// stay inside the window (true for the faces adjacent to the centre cell).
template <int V, int ND>
__device__ __forceinline__ float face_n0sq(const Window<V, ND>& w, int A, int qz, int qy, int qx, int s) {
  const int ez = (A == 2), ey = (A == 1), ex = (A == 0);
  const float lo = w.c[qz][qy][qx][s], hi = w.c[qz + ez][qy + ey][qx + ex][s];
  const float dd = hi - lo;
  float n0 = dd * dd;
  const float m0 = 0.5f * (hi + lo);
#pragma unroll
  for (int T = 0; T < ND; ++T) {
    if (T == A) continue;
    const int tz = (T == 2), ty = (T == 1), tx = (T == 0);
    const float mp = 0.5f * (w.c[qz + ez + tz][qy + ey + ty][qx + ex + tx][s] + w.c[qz + tz][qy + ty][qx + tx][s]);
    const float mm = 0.5f * (w.c[qz + ez - tz][qy + ey - ty][qx + ex - tx][s] + w.c[qz - tz][qy - ty][qx - tx][s]);
    const float a = mp - m0, b = m0 - mm;
    n0 = fmaf(0.5f * a, a, n0);
    n0 = fmaf(0.5f * b, b, n0);
  }
  return n0;
}

// The same N0^2 for slice lanes (2h, 2h+1) at once with Blackwell's packed fp32x2 instructions (FFMA2 /
// FADD2 / FMUL2, sm_100): the stencil kernels are bound by instruction issue, not by the FMA pipe, and a
// packed instruction does two lanes' worth of arithmetic in one issue slot. Operation for operation the
// same roundings as face_n0sq() (a - b is formed as fma(b, -1, a), which rounds identically).
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.0f, -1.0f), a); }

template <int V, int ND>
__device__ __forceinline__ float2 face_n0sq2(const Window<V, ND>& w, int A, int qz, int qy, int qx, int h) {
  const int ez = (A == 2), ey = (A == 1), ex = (A == 0);
  const float2 half = make_float2(0.5f, 0.5f);
#define W2(z, y, x) make_float2(w.c[z][y][x][2 * h], w.c[z][y][x][2 * h + 1])
  const float2 lo = W2(qz, qy, qx), hi = W2(qz + ez, qy + ey, qx + ex);
  const float2 dd = sub2(hi, lo);
  float2 n0 = __fmul2_rn(dd, dd);
  const float2 m0 = __fmul2_rn(half, __fadd2_rn(hi, lo));
#pragma unroll
  for (int T = 0; T < ND; ++T) {
    if (T == A) continue;
    const int tz = (T == 2), ty = (T == 1), tx = (T == 0);
    const float2 mp = __fmul2_rn(half, __fadd2_rn(W2(qz + ez + tz, qy + ey + ty, qx + ex + tx), W2(qz + tz, qy + ty, qx + tx)));
    const float2 mm = __fmul2_rn(half, __fadd2_rn(W2(qz + ez - tz, qy + ey - ty, qx + ex - tx), W2(qz - tz, qy - ty, qx - tx)));
    const float2 a = sub2(mp, m0), b = sub2(m0, mm);
    n0 = __ffma2_rn(__fmul2_rn(half, a), a, n0);
    n0 = __ffma2_rn(__fmul2_rn(half, b), b, n0);
  }
#undef W2
  return n0;
}

// thread -> voxel mapping shared by all stencil kernels: block (32,4), grid (nx/32, ny/(4 rows) * nz, G);
// a block sweeps `rows` groups of 4 image rows (rr = 0..rows-1; chosen by tv_rows() so that the grid still
// fills the GPU), so that its fixed costs - zeroing and
// flushing a shared histogram, a block-wide reduction of fp64 sums - are paid once per 32 x 4 rows voxels
// (they were most of the instructions of these kernels when a block handled 32 x 4 voxels only: 4.1 -> 3.05 ms
// of TV work per outer iteration at c4)
struct Vox {
  int i, j, k, g, tid;
  bool active;
  unsigned blk, nblk;
};
__device__ __forceinline__ Vox vox_of_thread(const Dims& d, int rr, int rows, int br = 4) {
  Vox v;
  const int nby = (d.ny + br * rows - 1) / (br * rows);
  v.i = blockIdx.x * 32 + threadIdx.x;
  v.k = blockIdx.y / nby;
  v.j = ((blockIdx.y - v.k * nby) * rows + rr) * br + threadIdx.y;
  v.g = blockIdx.z;
  v.tid = threadIdx.y * 32 + threadIdx.x;
  v.active = v.i < d.nx && v.j < d.ny;
  v.blk = blockIdx.y * gridDim.x + blockIdx.x;
  v.nblk = gridDim.x * gridDim.y;
  return v;
}
static dim3 vox_grid(const Dims& d, int rows, int br = 4) {
  return dim3((d.nx + 31) / 32, ((d.ny + br * rows - 1) / (br * rows)) * d.nz, d.G);
}
// A volume is ONE group: its blocks' partial sums are finished by a single block and every block pays the fixed
// costs above, so a 3D block sweeps up to TV_ROWS3D row groups instead of 8 / 16 (c5: 16 384-32 768 blocks otherwise)
#ifndef TV_ROWS3D
#define TV_ROWS3D 32 /* c5 TV per outer iteration: 11.0 / 10.0 / 9.7 / 9.9 / 11.2 ms for 8 / 16 / 32 / 48 / 64 */
#endif
#define TV_MAXROWS(d, n2d) ((d).ndim == 3 ? TV_ROWS3D : (n2d))
// row groups per block: as many as leave at least ~16 blocks per SM (8 for the 256-thread trial kernel)
static int tv_rows(const Dims& d, int rows_per_group, int max_rows, int min_blocks) {
  const long long blocks = (long long)((d.nx + 31) / 32) * ((d.ny + rows_per_group - 1) / rows_per_group) * d.nz * d.G;
  long long r = blocks / min_blocks;
  if (r < 1) r = 1;
  if (r > max_rows) r = max_rows;
  return (int)r;
}

// ---------------------------------------------------------------------------------------------
// a4.1  faces: N0^2 of the ND faces owned by each voxel (towards +x, +y, +z) -> n0 planes, plus the
// first radix pass (top 11 of the 31 value bits) of the per-slice histogram over INTERIOR faces.
// Exact zeros (flat regions) are counted with a ballot instead of hammering one shared bin.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void hist_add(unsigned* hist_s, unsigned bits, int shift, unsigned mask, bool valid) {
  const unsigned bin = (bits >> shift) & mask;
  const bool zero = valid && bin == 0;
  const unsigned zb = __ballot_sync(0xffffffffu, zero);
  if (valid && bin != 0) atomicAdd(&hist_s[bin], 1u);
  if ((threadIdx.x & 31) == 0 && zb) atomicAdd(&hist_s[0], (unsigned)__popc(zb));
}

template <int V, int ND>
__global__ void __launch_bounds__(128, TV_FMINB) k_tv_faces(Dims d, int rows, const float* __restrict__ f, float* __restrict__ n0,
                                                  unsigned* __restrict__ hist) {
  __shared__ unsigned hs[V][2048];
  const int tid0 = threadIdx.y * 32 + threadIdx.x;
  for (int t = tid0; t < V * 2048; t += 128) (&hs[0][0])[t] = 0;
  __syncthreads();
  const int lim[3] = {d.nx - 1, d.ny - 1, d.nz - 1};
  for (int rr = 0; rr < rows; ++rr) {
  const Vox p = vox_of_thread(d, rr, rows);
  const int pos[3] = {p.i, p.j, p.k};
  float val[ND][V];
  if (p.active) {
    Window<V, ND> w;
    load_window<V, ND>(d, f, p.g, p.i, p.j, p.k, w);
    const int cz = (ND == 3) ? 1 : 0;
#pragma unroll
    for (int A = 0; A < ND; ++A) {
      if (V % 2 == 0) {
#pragma unroll
        for (int hh = 0; hh < V / 2; ++hh) {
          const float2 t = face_n0sq2<V, ND>(w, A, cz, 1, 1, hh);
          val[A][2 * hh] = pos[A] < lim[A] ? t.x : 0.0f;
          val[A][2 * hh + (V > 1)] = pos[A] < lim[A] ? t.y : 0.0f;
        }
      } else {
#pragma unroll
        for (int s = 0; s < V; ++s) val[A][s] = pos[A] < lim[A] ? face_n0sq<V, ND>(w, A, cz, 1, 1, s) : 0.0f;
      }
    }
    const size_t e = (size_t)p.g * d.npix + ((size_t)p.k * d.ny + p.j) * d.nx + p.i;
#pragma unroll
    for (int A = 0; A < ND; ++A) Pack<V>::st(n0 + (size_t)A * d.G * d.npix * V, e, val[A]);
  }
#pragma unroll
  for (int A = 0; A < ND; ++A) {
    const bool valid = p.active && pos[A] < lim[A];
#pragma unroll
    for (int s = 0; s < V; ++s) hist_add(hs[s], valid ? __float_as_uint(val[A][s]) : 0u, 20, 2047u, valid);
  }
  }  // rr
  __syncthreads();
  for (int t = tid0; t < V * 2048; t += 128) {
    const unsigned c = (&hs[0][0])[t];
    if (c) atomicAdd(&hist[(size_t)(blockIdx.z * V + t / 2048) * 2048 + (t & 2047)], c);
  }
}

// a4.2  later radix passes over the stored N0^2 planes: only values whose higher bits equal the
// prefix found so far are counted.
template <int V, int ND>
__global__ void __launch_bounds__(128) k_tv_hist(Dims d, int rows, const float* __restrict__ n0, unsigned* __restrict__ hist,
                                                 Scal sc, int shift, unsigned mask, int prefix_shift) {
  __shared__ unsigned hs[V][1024];
  const int tid0 = threadIdx.y * 32 + threadIdx.x;
  for (int t = tid0; t < V * 1024; t += 128) (&hs[0][0])[t] = 0;
  __syncthreads();
  const int lim[3] = {d.nx - 1, d.ny - 1, d.nz - 1};
  unsigned pre[V];
#pragma unroll
  for (int s = 0; s < V; ++s) pre[s] = sc.sel_prefix[blockIdx.z * V + s] >> prefix_shift;
  for (int rr = 0; rr < rows; ++rr) {
  const Vox p = vox_of_thread(d, rr, rows);
  const int pos[3] = {p.i, p.j, p.k};
  const size_t e = (size_t)p.g * d.npix + ((size_t)p.k * d.ny + p.j) * d.nx + p.i;
#pragma unroll
  for (int A = 0; A < ND; ++A) {
    float val[V];
    const bool inside = p.active && pos[A] < lim[A];
    if (inside) Pack<V>::ldcg(n0 + (size_t)A * d.G * d.npix * V, e, val);
    unsigned bits[V];
    bool valid[V], anyv = false;
#pragma unroll
    for (int s = 0; s < V; ++s) {
      bits[s] = inside ? __float_as_uint(val[s]) : 0u;
      valid[s] = inside && (bits[s] >> prefix_shift) == pre[s];
      anyv |= valid[s];
    }
    // only a small fraction of the values carries the prefix found so far: most warps have nothing to add
    if (!__any_sync(0xffffffffu, anyv)) continue;
#pragma unroll
    for (int s = 0; s < V; ++s) hist_add(hs[s], bits[s], shift, mask, valid[s]);
  }
  }  // rr
  __syncthreads();
  for (int t = tid0; t < V * 1024; t += 128) {
    const unsigned c = (&hs[0][0])[t];
    if (c) atomicAdd(&hist[(size_t)(blockIdx.z * V + t / 1024) * 2048 + (t & 1023)], c);
  }
}

// a4.3  per slice: find the bin holding the element of rank sel_rank, extend the prefix, clear the
// histogram. After the last pass the prefix IS the bit pattern of the k-th smallest N0^2 (O6).
// Fused path (lists != 0): after the first pass the slice is a HIT when the bin found lies within one bin of the
// prediction (so every value of that bin is in the candidate list), no staging buffer overflowed and the list
// fits; after the final pass the bin becomes the next sweep's prediction and the list is emptied.
__global__ void __launch_bounds__(256) k_tv_select(Scal sc, unsigned* __restrict__ hist, int nbins, int shift,
                                                   int first, int final_pass, unsigned long long rank0, float eps2,
                                                   StatRing ring, int lists, unsigned cand_cap, int pos = 0, int gv = 0) {
  __shared__ unsigned tot[256];
  __shared__ unsigned found_bin, found_before;
  const int sl = blockIdx.x, t = threadIdx.x;
  if (gv > 0) {
    // first pass after k_tv_scan1f: the full histogram exists only for groups (gv slices) in which a slice missed
    bool allhit = true;
    for (int s = 0; s < gv; ++s) allhit = allhit && sc.fhit[(sl / gv) * gv + s] != 0;
    if (allhit) return;
  }
  unsigned* h = hist + (size_t)sl * 2048;
  const int per = nbins / 256;  // 8 or 4
  unsigned loc[8], sum = 0;
  for (int q = 0; q < per; ++q) { loc[q] = h[t * per + q]; sum += loc[q]; }
  tot[t] = sum;
  __syncthreads();
  // inclusive scan over the 256 thread totals (Hillis-Steele; tiny)
  for (int o = 1; o < 256; o <<= 1) {
    unsigned add = t >= o ? tot[t - o] : 0u;
    __syncthreads();
    tot[t] += add;
    __syncthreads();
  }
  const unsigned rank = first ? (unsigned)rank0 : sc.sel_rank[sl];
  const unsigned before = tot[t] - sum;
  if (rank > before && rank <= tot[t]) {
    unsigned cum = before;
    for (int q = 0; q < per; ++q) {
      if (rank <= cum + loc[q]) { found_bin = t * per + q; found_before = cum; break; }
      cum += loc[q];
    }
  }
  __syncthreads();
  for (int q = 0; q < per; ++q) h[t * per + q] = 0;
  if (t == 0) {
    const unsigned prefix = (first ? 0u : sc.sel_prefix[sl]) | (found_bin << shift);
    sc.sel_prefix[sl] = prefix;
    sc.sel_rank[sl] = rank - found_before;
    if (lists && first) {
      const int dbin = (int)found_bin - sc.pred[sl];
      sc.hit[sl] = (dbin >= -1 && dbin <= 1 && sc.ovf[sl] == 0u && sc.cand_cnt[sl] <= cand_cap) ? 1 : 0;
    }
    if (final_pass) {
      const float s2 = fmaxf(__uint_as_float(prefix), eps2);
      sc.sigma2[sl] = s2;
      ring.slot()[sl].sigma = sqrt((double)s2);
      if (lists) {
        // prediction for the next sweep: this bin; across Step 1 (pos bit 1: this is the last sweep of the outer
        // iteration) this bin plus the jump the previous Step 1 caused (measured in the first sweep after it, pos bit 0)
        const int bin = (int)(prefix >> 20);
        if ((pos & 1) && sc.lastbin[sl] >= 0) sc.jump[sl] = max(-64, min(64, bin - sc.lastbin[sl]));
        if (pos & 2) sc.lastbin[sl] = bin;
        sc.pred[sl] = (pos & 2) ? bin + sc.jump[sl] : bin;
        sc.cand_cnt[sl] = 0u;
        sc.ovf[sl] = 0u;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Fused sigma selection (ctr_reconstruct): no N0^2 planes. The face magnitudes are recomputed from the L1-cached
// window wherever they are needed (4 B per voxel read instead of 8 B written + 8 B read back per pass), and
// the second and third radix passes run on a CANDIDATE LIST instead of the image: sigma moves little from one
// sweep to the next, so the first pass appends every value whose top 11 bits lie within one bin of the bin the
// previous sweep found (a few per cent of the faces) to a per-slice list - staged per block in shared memory,
// one global atomicAdd per block and slice - and if the winning bin is indeed covered (k_tv_select: HIT), passes
// 2 and 3 only filter that list. On a MISS (first sweep, or sigma jumped) the blocks of k_tv_scan23 recompute the
// magnitudes from the image instead: same counts, so sigma is the exact order statistic either way (O6).
// ---------------------------------------------------------------------------------------------
#define TV_SCAP(V) (3072 / (V)) /* staging entries per block and slice (a block sees 32 x 8 x rows voxels x ND faces per slice) */
#ifndef TV_SMINB
#define TV_SMINB 3
#endif
#ifndef TV_FAST_SCAN
#define TV_FAST_SCAN 1
#endif
#ifndef TV_SFMINB
#define TV_SFMINB 5 /* min blocks per SM of k_tv_scan1f (c4 TV per outer iteration: 1.96 / 1.92 / 1.91 / 1.91 ms for 3 / 4 / 5 / 6) */
#endif

template <int V, int ND>
__device__ __forceinline__ void own_face_values(const Dims& d, const Window<V, ND>& w, const int (&pos)[3],
                                                const int (&lim)[3], float (&val)[ND][V]) {
  const int cz = (ND == 3) ? 1 : 0;
#pragma unroll
  for (int A = 0; A < ND; ++A) {
    if (V % 2 == 0) {
#pragma unroll
      for (int hh = 0; hh < V / 2; ++hh) {
        const float2 t = face_n0sq2<V, ND>(w, A, cz, 1, 1, hh);
        val[A][2 * hh] = pos[A] < lim[A] ? t.x : 0.0f;
        val[A][2 * hh + (V > 1)] = pos[A] < lim[A] ? t.y : 0.0f;
      }
    } else {
#pragma unroll
      for (int s = 0; s < V; ++s) val[A][s] = pos[A] < lim[A] ? face_n0sq<V, ND>(w, A, cz, 1, 1, s) : 0.0f;
    }
  }
  (void)d;
}

template <int V, int ND>
__global__ void __launch_bounds__(256, TV_SMINB) k_tv_scan1(Dims d, int rows, const float* __restrict__ f,
                                                            unsigned* __restrict__ hist, Scal sc,
                                                            unsigned* __restrict__ cand, unsigned cap, int after_fast) {
  __shared__ unsigned hs[V][2048];
  __shared__ unsigned stage[V][TV_SCAP(V)];
  __shared__ unsigned stage_n[V], stage_base[V];
  const int tid0 = threadIdx.y * 32 + threadIdx.x;
  for (int t = tid0; t < V * 2048; t += 256) (&hs[0][0])[t] = 0;
  if (tid0 < V) stage_n[tid0] = 0;
  int pred[V];
  bool need = !after_fast;
#pragma unroll
  for (int s = 0; s < V; ++s) {
    pred[s] = sc.pred[blockIdx.z * V + s];
    if (after_fast) {
      // after k_tv_scan1f: only groups with a slice that missed need the full histogram, and the slices that hit
      // keep the candidate lists they have (a prediction that can never match stops a second append)
      const bool fh = sc.fhit[blockIdx.z * V + s] != 0;
      need = need || !fh;
      if (fh) pred[s] = INT_MIN / 2;
    }
  }
  if (!need) return;
  __syncthreads();
  const int lim[3] = {d.nx - 1, d.ny - 1, d.nz - 1};
  unsigned nzero[V];  // exact zeros (flat regions) are counted in a register instead of hammering bin 0
#pragma unroll
  for (int s = 0; s < V; ++s) nzero[s] = 0u;
  for (int rr = 0; rr < rows; ++rr) {
    const Vox p = vox_of_thread(d, rr, rows, 8);
    const int pos[3] = {p.i, p.j, p.k};
    if (!p.active) continue;
    float val[ND][V];
    Window<V, ND> w;
    load_window<V, ND>(d, f, p.g, p.i, p.j, p.k, w);
    own_face_values<V, ND>(d, w, pos, lim, val);
#pragma unroll
    for (int A = 0; A < ND; ++A) {
      if (pos[A] >= lim[A]) continue;  // border face
#pragma unroll
      for (int s = 0; s < V; ++s) {
        const unsigned bits = __float_as_uint(val[A][s]);
        const unsigned bin = bits >> 20;
        if (bin) atomicAdd(&hs[s][bin], 1u);
        else ++nzero[s];
        if (bin + 1u - (unsigned)pred[s] <= 2u) {  // |bin - pred| <= 1 (pred < 0 never matches)
          const unsigned at = atomicAdd(&stage_n[s], 1u);
          if (at < TV_SCAP(V)) stage[s][at] = bits;
        }
      }
    }
  }
#pragma unroll
  for (int s = 0; s < V; ++s) {
    const unsigned z = __reduce_add_sync(0xffffffffu, nzero[s]);
    if ((threadIdx.x & 31) == 0 && z) atomicAdd(&hs[s][0], z);
  }
  __syncthreads();
  for (int t = tid0; t < V * 2048; t += 256) {
    const unsigned c = (&hs[0][0])[t];
    if (c) atomicAdd(&hist[(size_t)(blockIdx.z * V + t / 2048) * 2048 + (t & 2047)], c);
  }
  if (tid0 < V) {
    const int sl = blockIdx.z * V + tid0;
    unsigned n = stage_n[tid0];
    if (n > TV_SCAP(V)) { atomicOr(&sc.ovf[sl], 1u); n = TV_SCAP(V); }
    stage_n[tid0] = n;
    stage_base[tid0] = n ? atomicAdd(&sc.cand_cnt[sl], n) : 0u;
  }
  __syncthreads();
#pragma unroll
  for (int s = 0; s < V; ++s) {
    const unsigned n = stage_n[s], base = stage_base[s];
    unsigned* dst = cand + (size_t)(blockIdx.z * V + s) * cap;
    for (unsigned t = tid0; t < n; t += 256)
      if (base + t < cap) dst[base + t] = stage[s][t];
  }
}

// Fast first pass (large problems, steady state): the winning bin is almost always within one bin of the prediction,
// and then all the first pass has to deliver is the number of values BELOW the three-bin window, the counts of the
// three bins and the candidate list - no 2048-bin histogram, i.e. no shared-memory atomic per value (ncu: half of
// k_tv_scan1's instructions are the integer and branch work around them). hist[sl][0] = below, [1..3] = the window bins.
// k_tv_select_f takes the decision; a slice whose rank falls outside the window (or whose list overflowed) is a MISS,
// and its group then runs the full k_tv_scan1 / k_tv_select pass: sigma is the exact order statistic either way.
template <int V, int ND>
__global__ void __launch_bounds__(256, TV_SFMINB) k_tv_scan1f(Dims d, int rows, const float* __restrict__ f,
                                                             unsigned* __restrict__ hist, Scal sc,
                                                             unsigned* __restrict__ cand, unsigned cap) {
  __shared__ unsigned cnt_s[V][4];
  __shared__ unsigned stage[V][TV_SCAP(V)];
  __shared__ unsigned stage_n[V], stage_base[V];
  const int tid0 = threadIdx.y * 32 + threadIdx.x;
  if (tid0 < V * 4) (&cnt_s[0][0])[tid0] = 0;
  if (tid0 < V) stage_n[tid0] = 0;
  int lo[V];
#pragma unroll
  for (int s = 0; s < V; ++s) lo[s] = sc.pred[blockIdx.z * V + s] - 1;  // no prediction: hugely negative, nothing matches
  __syncthreads();
  const int lim[3] = {d.nx - 1, d.ny - 1, d.nz - 1};
  unsigned nbelow[V];
#pragma unroll
  for (int s = 0; s < V; ++s) nbelow[s] = 0u;
  for (int rr = 0; rr < rows; ++rr) {
    const Vox p = vox_of_thread(d, rr, rows, 8);
    const int pos[3] = {p.i, p.j, p.k};
    if (!p.active) continue;
    float val[ND][V];
    Window<V, ND> w;
    load_window<V, ND>(d, f, p.g, p.i, p.j, p.k, w);
    own_face_values<V, ND>(d, w, pos, lim, val);
#pragma unroll
    for (int A = 0; A < ND; ++A) {
      if (pos[A] >= lim[A]) continue;  // border face
#pragma unroll
      for (int s = 0; s < V; ++s) {
        const unsigned bits = __float_as_uint(val[A][s]);
        const int bin = (int)(bits >> 20);
        nbelow[s] += bin < lo[s] ? 1u : 0u;
        const unsigned rel = (unsigned)(bin - lo[s]);
        if (rel < 3u) {
          atomicAdd(&cnt_s[s][1 + rel], 1u);
          const unsigned at = atomicAdd(&stage_n[s], 1u);
          if (at < TV_SCAP(V)) stage[s][at] = bits;
        }
      }
    }
  }
#pragma unroll
  for (int s = 0; s < V; ++s) {
    const unsigned z = __reduce_add_sync(0xffffffffu, nbelow[s]);
    if ((threadIdx.x & 31) == 0 && z) atomicAdd(&cnt_s[s][0], z);
  }
  __syncthreads();
  if (tid0 < V * 4) {
    const unsigned c = (&cnt_s[0][0])[tid0];
    if (c) atomicAdd(&hist[(size_t)(blockIdx.z * V + tid0 / 4) * 2048 + (tid0 & 3)], c);
  }
  if (tid0 < V) {
    const int sl = blockIdx.z * V + tid0;
    unsigned n = stage_n[tid0];
    if (n > TV_SCAP(V)) { atomicOr(&sc.ovf[sl], 1u); n = TV_SCAP(V); }
    stage_n[tid0] = n;
    stage_base[tid0] = n ? atomicAdd(&sc.cand_cnt[sl], n) : 0u;
  }
  __syncthreads();
#pragma unroll
  for (int s = 0; s < V; ++s) {
    const unsigned n = stage_n[s], base = stage_base[s];
    unsigned* dst = cand + (size_t)(blockIdx.z * V + s) * cap;
    for (unsigned t = tid0; t < n; t += 256)
      if (base + t < cap) dst[base + t] = stage[s][t];
  }
}

// decision of the fast first pass, one thread per slice
__global__ void __launch_bounds__(128) k_tv_select_f(Scal sc, unsigned* __restrict__ hist, int Bp, unsigned long long rank0,
                                                     unsigned cand_cap) {
  const int sl = blockIdx.x * 128 + threadIdx.x;
  if (sl >= Bp) return;
  unsigned* h = hist + (size_t)sl * 2048;
  const unsigned below = h[0], c[3] = {h[1], h[2], h[3]};
  h[0] = 0u; h[1] = 0u; h[2] = 0u; h[3] = 0u;
  const unsigned rank = (unsigned)rank0;
  const int lo = sc.pred[sl] - 1;
  const bool ok = sc.ovf[sl] == 0u && sc.cand_cnt[sl] <= cand_cap && rank > below && rank <= below + c[0] + c[1] + c[2];
  if (ok) {
    unsigned cum = below;
    int j = 0;
    while (rank > cum + c[j]) { cum += c[j]; ++j; }
    sc.sel_prefix[sl] = (unsigned)(lo + j) << 20;
    sc.sel_rank[sl] = rank - cum;
    sc.hit[sl] = 1;
    sc.fhit[sl] = 1;
  } else {
    sc.fhit[sl] = 0;
    sc.cand_cnt[sl] = 0u;  // the full pass fills the list again
    sc.ovf[sl] = 0u;
  }
}

// passes 2 and 3 of the fused selection: histogram of the next bits of the values that carry the prefix found
// so far; from the candidate lists when every slice of the group was a hit, from the image otherwise
template <int V, int ND>
__global__ void __launch_bounds__(256, TV_SMINB) k_tv_scan23(Dims d, int rows, const float* __restrict__ f,
                                                             unsigned* __restrict__ hist, Scal sc,
                                                             const unsigned* __restrict__ cand, unsigned cap, int shift,
                                                             unsigned mask, int prefix_shift) {
  __shared__ unsigned hs[V][1024];
  const int tid0 = threadIdx.y * 32 + threadIdx.x;
  bool hit = true;
  unsigned pre[V], cnt[V], maxc = 0;
#pragma unroll
  for (int s = 0; s < V; ++s) {
    const int sl = blockIdx.z * V + s;
    hit = hit && sc.hit[sl] != 0;
    pre[s] = sc.sel_prefix[sl] >> prefix_shift;
    cnt[s] = sc.cand_cnt[sl];
    maxc = max(maxc, cnt[s]);
  }
  const unsigned blk = blockIdx.y * gridDim.x + blockIdx.x, nblk = gridDim.x * gridDim.y;
  if (hit && blk * 256u >= maxc) return;  // nothing of the lists falls to this block
  for (int t = tid0; t < V * 1024; t += 256) (&hs[0][0])[t] = 0;
  __syncthreads();
  if (hit) {
#pragma unroll
    for (int s = 0; s < V; ++s) {
      const unsigned* src = cand + (size_t)(blockIdx.z * V + s) * cap;
      for (unsigned e = blk * 256u + tid0; e < cnt[s]; e += nblk * 256u) {
        const unsigned bits = __ldcg(src + e);
        if ((bits >> prefix_shift) == pre[s]) atomicAdd(&hs[s][(bits >> shift) & mask], 1u);
      }
    }
  } else {
    const int lim[3] = {d.nx - 1, d.ny - 1, d.nz - 1};
    for (int rr = 0; rr < rows; ++rr) {
      const Vox p = vox_of_thread(d, rr, rows, 8);
      const int pos[3] = {p.i, p.j, p.k};
      float val[ND][V];
      if (p.active) {
        Window<V, ND> w;
        load_window<V, ND>(d, f, p.g, p.i, p.j, p.k, w);
        own_face_values<V, ND>(d, w, pos, lim, val);
      }
#pragma unroll
      for (int A = 0; A < ND; ++A) {
        const bool inside = p.active && pos[A] < lim[A];
        unsigned bits[V];
        bool valid[V], anyv = false;
#pragma unroll
        for (int s = 0; s < V; ++s) {
          bits[s] = inside ? __float_as_uint(val[A][s]) : 0u;
          valid[s] = inside && (bits[s] >> prefix_shift) == pre[s];
          anyv |= valid[s];
        }
        if (!__any_sync(0xffffffffu, anyv)) continue;
#pragma unroll
        for (int s = 0; s < V; ++s) hist_add(hs[s], bits[s], shift, mask, valid[s]);
      }
    }
  }
  __syncthreads();
  for (int t = tid0; t < V * 1024; t += 256) {
    const unsigned c = (&hs[0][0])[t];
    if (c) atomicAdd(&hist[(size_t)(blockIdx.z * V + t / 1024) * 2048 + (t & 1023)], c);
  }
}

// a4.4  w = exp(-N0^2/sigma^2) on interior faces, 0 on border faces; TV mode: 1
template <int V, int ND>
__global__ void __launch_bounds__(128) k_tv_weights(Dims d, int rows, const float* __restrict__ n0, float* __restrict__ w,
                                                    Scal sc, int mode, StatRing ring) {
  if (mode == 1 && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0 && threadIdx.y == 0) {
#pragma unroll
    for (int s = 0; s < V; ++s) ring.slot()[blockIdx.z * V + s].sigma = 0.0;  // plain TV: no sigma (documented as 0)
  }
  float inv[V];
#pragma unroll
  for (int s = 0; s < V; ++s) inv[s] = -1.0f / sc.sigma2[blockIdx.z * V + s];
  for (int rr = 0; rr < rows; ++rr) {
  const Vox p = vox_of_thread(d, rr, rows);
  if (!p.active) continue;
  const int lim[3] = {d.nx - 1, d.ny - 1, d.nz - 1};
  const int pos[3] = {p.i, p.j, p.k};
  const size_t e = (size_t)p.g * d.npix + ((size_t)p.k * d.ny + p.j) * d.nx + p.i;
#pragma unroll
  for (int A = 0; A < ND; ++A) {
    float val[V], o[V];
    Pack<V>::ldcg(n0 + (size_t)A * d.G * d.npix * V, e, val);
#pragma unroll
    for (int s = 0; s < V; ++s) o[s] = pos[A] < lim[A] ? (mode == 1 ? 1.0f : expf(val[s] * inv[s])) : 0.0f;
    Pack<V>::st(w + (size_t)A * d.G * d.npix * V, e, o);
  }
  }  // rr
}

// ---------------------------------------------------------------------------------------------
// a5  gradient g = lambda (f - v) - sum_A (flux_A(p) - flux_A(p - e_A)),
//     flux_A = w_A d_A / sqrt(N0^2 + eps^2) (A2), plus G = ||g||^2 and E0 (O9).
// ---------------------------------------------------------------------------------------------
// WSRC = 0: the weights come from the caller's planes w (ctr_eptv_step: they need not belong to this x);
// WSRC = 1: fused path of ctr_reconstruct, w = exp(-N0^2/sigma^2) (A3) is evaluated on the fly
// from the magnitudes of THIS f and the sigma^2 the selection has just left in sc.sigma2 (TV mode: w = 1): no
// weight planes, no magnitude planes. Either way N0^2 of the four (six) faces of a voxel is recomputed from its
// window: all their stencils lie inside it.
// w = exp(-N0^2/sigma^2) = 2^(N0^2 k), k = -log2(e)/sigma^2 formed once per block: one FMUL and one MUFU.EX2 per
// face (__expf adds a denormal-range fix-up per call; w underflowing to 0 for N0 >> sigma is what is wanted)
__device__ __forceinline__ float edge_weight(float n0sq, float k) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(n0sq * k));
  return r;
}
#define CTR_LOG2E 1.4426950408889634f
// one MUFU.RSQ, no denormal fix-up: the arguments are N0^2 + eps^2 (1e-8 with the default eps); callers treat
// anything below 1e-30 as a flat face
__device__ __forceinline__ float rsqrt_fast(float x) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

template <int V, int ND, int WSRC>
__global__ void __launch_bounds__(128, TV_GMINB) k_tv_gradient(Dims d, int rows, const float* __restrict__ f, const float* __restrict__ v,
                                                     const float* __restrict__ w, float* __restrict__ gout, TvParams tp,
                                                     Scal sc, double* part, unsigned* counter, StatRing ring) {
  // per-thread sums over its (at most 8) voxels in fp32, everything above that in fp64
  float acc[2 * V];
#pragma unroll
  for (int s = 0; s < 2 * V; ++s) acc[s] = 0.0f;
  float nis2[V];
#pragma unroll
  for (int s = 0; s < V; ++s) nis2[s] = WSRC ? -CTR_LOG2E / sc.sigma2[blockIdx.z * V + s] : 0.0f;
  const int lim[3] = {d.nx - 1, d.ny - 1, d.nz - 1};
  for (int rr = 0; rr < rows; ++rr) {
  const Vox p = vox_of_thread(d, rr, rows);
  if (p.active) {
    Window<V, ND> win;
    load_window<V, ND>(d, f, p.g, p.i, p.j, p.k, win);
    const int cz = (ND == 3) ? 1 : 0;
    const int pos[3] = {p.i, p.j, p.k};
    const size_t stride[3] = {1, (size_t)d.nx, (size_t)d.nx * d.ny};
    const size_t e = (size_t)p.g * d.npix + ((size_t)p.k * d.ny + p.j) * d.nx + p.i;
    const size_t plane = (size_t)d.G * d.npix * V;
    const float eps2 = tp.eps * tp.eps;
    float vv[V], gv[V], etv[V];
    Pack<V>::ldcg(v, e, vv);
#pragma unroll
    for (int s = 0; s < V; ++s) {
      gv[s] = tp.lambda * (win.c[cz][1][1][s] - vv[s]);
      etv[s] = 0.0f;
    }
#pragma unroll
    for (int A = 0; A < ND; ++A) {
      float wp[V], wm[V];
      if (!WSRC) {
        Pack<V>::ldcg(w + A * plane, e, wp);  // border faces store 0
        if (pos[A] > 0) Pack<V>::ldcg(w + A * plane, e - stride[A], wm);
        else {
#pragma unroll
          for (int s = 0; s < V; ++s) wm[s] = 0.0f;
        }
      }
      const int ez = (A == 2), ey = (A == 1), ex = (A == 0);
      float rp[V], rm[V];  // raw N0^2 of the face towards +A (owned by this voxel) and towards -A (owned by the neighbour)
      if (V % 2 == 0) {
#pragma unroll
        for (int hh = 0; hh < V / 2; ++hh) {
          const float2 a = face_n0sq2<V, ND>(win, A, cz, 1, 1, hh), b = face_n0sq2<V, ND>(win, A, cz - ez, 1 - ey, 1 - ex, hh);
          rp[2 * hh] = a.x; rp[2 * hh + (V > 1)] = a.y;
          rm[2 * hh] = b.x; rm[2 * hh + (V > 1)] = b.y;
        }
      } else {
#pragma unroll
        for (int s = 0; s < V; ++s) {
          rp[s] = face_n0sq<V, ND>(win, A, cz, 1, 1, s);
          rm[s] = face_n0sq<V, ND>(win, A, cz - ez, 1 - ey, 1 - ex, s);
        }
      }
      // border faces: the face towards -A of the first voxel has dm = 0 exactly (replicated neighbour), so only
      // the +A face of the last voxel needs its weight masked (it would otherwise enter the energy)
      const float maskp = pos[A] < lim[A] ? 1.0f : 0.0f;
#pragma unroll
      for (int s = 0; s < V; ++s) {
        if (WSRC) {
          wp[s] = tp.weights_mode == 1 ? maskp : maskp * edge_weight(rp[s], nis2[s]);
          wm[s] = tp.weights_mode == 1 ? 1.0f : edge_weight(rm[s], nis2[s]);
        }
        const float n0p = fmaxf(rp[s] + eps2, 1e-30f), n0m = fmaxf(rm[s] + eps2, 1e-30f);
        const float dp = win.c[cz + ez][1 + ey][1 + ex][s] - win.c[cz][1][1][s];
        const float dm = win.c[cz][1][1][s] - win.c[cz - ez][1 - ey][1 - ex][s];
        // sqrt(x) = x rsqrt(x): one special-function instruction per face serves both the flux and the energy
        const float ip = rsqrt_fast(n0p), im = rsqrt_fast(n0m);
        gv[s] -= wp[s] * dp * ip - wm[s] * dm * im;
        // (a flat face contributes exactly 0: north_star's invariant on a constant image)
        etv[s] = fmaf(wp[s], rp[s] > 0.0f ? fmaf(n0p, ip, -tp.eps) : 0.0f, etv[s]);
      }
    }
    Pack<V>::st(gout, e, gv);
#pragma unroll
    for (int s = 0; s < V; ++s) {
      const float df = win.c[cz][1][1][s] - vv[s];
      acc[s] = fmaf(gv[s], gv[s], acc[s]);
      acc[V + s] += fmaf(0.5f * tp.lambda * df, df, etv[s] * (1.0f / (float)ND));
    }
  }
  }  // rr
  double red[2 * V];
#pragma unroll
  for (int s = 0; s < 2 * V; ++s) red[s] = (double)acc[s];
  const Vox p = vox_of_thread(d, 0, rows);
  grid_reduce<2 * V>(red, part + (size_t)p.g * p.nblk * 2 * V, counter + p.g, p.nblk, p.blk, p.tid, 128,
                     [&](double(&sum)[2 * V]) {
#pragma unroll
                       for (int s = 0; s < V; ++s) {
                         const int sl = p.g * V + s;
                         sc.g2[sl] = sum[s];
                         sc.e0[sl] = sum[V + s];
                         sc.kacc[sl] = -1;
                         sc.tacc[sl] = 0.0f;
                         if (WSRC && tp.weights_mode == 1) ring.slot()[sl].sigma = 0.0;  // plain TV: no sigma
                       }
                     });
}

// ---------------------------------------------------------------------------------------------
// a6.1  Armijo trials, TV_KA candidates per pass.
// Along the search line every term of A3 is linear in t: the face magnitude of f - t g is
//   N0^2(t) = a - 2 t b + t^2 c,   a = N0^2(f), c = N0^2(g), b = the mixed form (same stencil),
// so (a, b, c) are formed once per face from differences of the f and g windows and each candidate
// costs two FMAs and a square root per face. The fidelity term is a quadratic in t with three
// candidate-independent sums: lambda/2 (D0 - 2 t D1 + t^2 D2), D0 = |f-v|^2, D1 = <f-v,g>, D2 = |g|^2.
// E(f - t_k g) with w frozen (O9) is assembled in fp64 by k_tv_trial_finish, which takes the first k with
// E <= E0 - c t_k |g|^2. Slices that accepted a step in an earlier pass are skipped.
// ---------------------------------------------------------------------------------------------
#ifndef TV_KA
#define TV_KA 8 /* candidates per pass; k <= 5 in every sweep seen, a later pass covers the rest (6 measured no faster) */
#endif

// the linear forms of A3 on the face between the centre cell and its +A neighbour,
// evaluated on windows wf and wg: returns a = sum c_i Lf_i^2, b = sum c_i Lf_i Lg_i, c = sum c_i Lg_i^2
template <int V, int ND>
__device__ __forceinline__ void face_forms(const Window<V, ND>& wf, const Window<V, ND>& wg, int A, int s, float& a,
                                           float& b, float& c) {
  const int cz = (ND == 3) ? 1 : 0;
  const int ez = (A == 2), ey = (A == 1), ex = (A == 0);
  const float df = wf.c[cz + ez][1 + ey][1 + ex][s] - wf.c[cz][1][1][s];
  const float dg = wg.c[cz + ez][1 + ey][1 + ex][s] - wg.c[cz][1][1][s];
  a = df * df; b = df * dg; c = dg * dg;
#pragma unroll
  for (int T = 0; T < ND; ++T) {
    if (T == A) continue;
    const int tz = (T == 2), ty = (T == 1), tx = (T == 0);
#pragma unroll
    for (int sg = -1; sg <= 1; sg += 2) {
      // m(+T) - m0 (sg = +1) or m0 - m(-T) (sg = -1), as half the sum of two differences
      const float lf = 0.5f * ((wf.c[cz + ez + sg * tz][1 + ey + sg * ty][1 + ex + sg * tx][s] - wf.c[cz + ez][1 + ey][1 + ex][s]) +
                               (wf.c[cz + sg * tz][1 + sg * ty][1 + sg * tx][s] - wf.c[cz][1][1][s]));
      const float lg = 0.5f * ((wg.c[cz + ez + sg * tz][1 + ey + sg * ty][1 + ex + sg * tx][s] - wg.c[cz + ez][1 + ey][1 + ex][s]) +
                               (wg.c[cz + sg * tz][1 + sg * ty][1 + sg * tx][s] - wg.c[cz][1][1][s]));
      a = fmaf(0.5f * lf, lf, a);
      b = fmaf(0.5f * lf, lg, b);
      c = fmaf(0.5f * lg, lg, c);
    }
  }
}

// face_forms() for slice lanes (2h, 2h+1) at once with packed fp32x2 instructions; same roundings per lane
template <int V, int ND>
__device__ __forceinline__ void face_forms2(const Window<V, ND>& wf, const Window<V, ND>& wg, int A, int h, float2& a,
                                            float2& b, float2& c) {
  const int cz = (ND == 3) ? 1 : 0;
  const int ez = (A == 2), ey = (A == 1), ex = (A == 0);
  const float2 half = make_float2(0.5f, 0.5f);
#define F2(w, z, y, x) make_float2(w.c[z][y][x][2 * h], w.c[z][y][x][2 * h + 1])
  const float2 df = sub2(F2(wf, cz + ez, 1 + ey, 1 + ex), F2(wf, cz, 1, 1));
  const float2 dg = sub2(F2(wg, cz + ez, 1 + ey, 1 + ex), F2(wg, cz, 1, 1));
  a = __fmul2_rn(df, df); b = __fmul2_rn(df, dg); c = __fmul2_rn(dg, dg);
#pragma unroll
  for (int T = 0; T < ND; ++T) {
    if (T == A) continue;
    const int tz = (T == 2), ty = (T == 1), tx = (T == 0);
#pragma unroll
    for (int sg = -1; sg <= 1; sg += 2) {
      const float2 lf = __fmul2_rn(half, __fadd2_rn(sub2(F2(wf, cz + ez + sg * tz, 1 + ey + sg * ty, 1 + ex + sg * tx), F2(wf, cz + ez, 1 + ey, 1 + ex)),
                                                   sub2(F2(wf, cz + sg * tz, 1 + sg * ty, 1 + sg * tx), F2(wf, cz, 1, 1))));
      const float2 lg = __fmul2_rn(half, __fadd2_rn(sub2(F2(wg, cz + ez + sg * tz, 1 + ey + sg * ty, 1 + ex + sg * tx), F2(wg, cz + ez, 1 + ey, 1 + ex)),
                                                   sub2(F2(wg, cz + sg * tz, 1 + sg * ty, 1 + sg * tx), F2(wg, cz, 1, 1))));
      const float2 hlf = __fmul2_rn(half, lf), hlg = __fmul2_rn(half, lg);
      a = __ffma2_rn(hlf, lf, a);
      b = __ffma2_rn(hlf, lg, b);
      c = __ffma2_rn(hlg, lg, c);
    }
  }
#undef F2
}

// block (32, 8); partials part[g][blk][NV], NV = TV_KA * V (TV energies, fp32 sums of one block's voxels
// widened to fp64) + 3 * V (D0, D1, D2 in fp64)
#ifndef TV_TW
#define TV_TW 4 /* warps (rows of 32 voxels) per block of the trial kernel; (4, 3) measured best of (4,3) (4,4) (8,2) */
#endif
#ifndef TV_TMINB
#define TV_TMINB 3
#endif
// WSRC as in k_tv_gradient: 0 = weight planes of the caller, 1 = w = exp(-N0^2(f)/sigma^2) on the fly (N0^2(f) is
// the form `a` below: the same stencil as face_n0sq(), differences taken in another order)
template <int V, int ND, int WSRC>
__global__ void __launch_bounds__(32 * TV_TW, TV_TMINB) k_tv_trial(Dims d, int rows, const float* __restrict__ f, const float* __restrict__ gin,
                                                  const float* __restrict__ v, const float* __restrict__ w, TvParams tp,
                                                  int k0, Scal sc, double* part) {
  constexpr int NE = TV_KA * V, NV = NE + 3 * V;
  __shared__ float colsum[TV_TW][32][33];
  __shared__ double wsum[TV_TW][NV];
  const int nby = (d.ny + TV_TW * rows - 1) / (TV_TW * rows);
  const int i = blockIdx.x * 32 + threadIdx.x;
  const int k = blockIdx.y / nby;
  const int g = blockIdx.z;
  const int lane = threadIdx.x, wid = threadIdx.y, tid = wid * 32 + lane;
  const unsigned blk = blockIdx.y * gridDim.x + blockIdx.x, nblk = gridDim.x * gridDim.y;
  bool todo[V], any = false;
#pragma unroll
  for (int s = 0; s < V; ++s) { todo[s] = sc.kacc[g * V + s] < 0; any |= todo[s]; }
  if (!any) return;
  float nis2[V];
#pragma unroll
  for (int s = 0; s < V; ++s) nis2[s] = WSRC ? -CTR_LOG2E / sc.sigma2[g * V + s] : 0.0f;
  const int lim[3] = {d.nx - 1, d.ny - 1, d.nz - 1};
  float et[NE];
  double dd[3 * V];
#pragma unroll
  for (int q = 0; q < NE; ++q) et[q] = 0.0f;
#pragma unroll
  for (int q = 0; q < 3 * V; ++q) dd[q] = 0.0;
  for (int rr = 0; rr < rows; ++rr) {  // a block sweeps `rows` groups of 8 rows: one reduction for all
  const int j = ((blockIdx.y - k * nby) * rows + rr) * TV_TW + threadIdx.y;
  const bool active = i < d.nx && j < d.ny;
  if (active) {
    Window<V, ND> wf, wg;
    load_window<V, ND>(d, f, g, i, j, k, wf);
    load_window<V, ND>(d, gin, g, i, j, k, wg);
    const int cz = (ND == 3) ? 1 : 0;
    const size_t e = (size_t)g * d.npix + ((size_t)k * d.ny + j) * d.nx + i;
    const size_t plane = (size_t)d.G * d.npix * V;
    const float eps = tp.eps, eps2 = tp.eps * tp.eps;
    const int pos[3] = {i, j, k};
    float vv[V];
    Pack<V>::ldcg(v, e, vv);
#pragma unroll
    for (int s = 0; s < V; ++s) {
      const float df = wf.c[cz][1][1][s] - vv[s], gg = wg.c[cz][1][1][s];
      dd[s] += (double)df * (double)df;
      dd[V + s] += (double)df * (double)gg;
      dd[2 * V + s] += (double)gg * (double)gg;
    }
    if (V % 2 == 0) {
      // packed path (V = 4): slice lanes in pairs, FFMA2 / FMUL2 throughout except max and rsqrt
      constexpr int H = V / 2 > 0 ? V / 2 : 1;
      float2 fa[ND][H], fb[ND][H], fc[ND][H], wA2[ND][H];
      const float2 eps22 = make_float2(eps2, eps2), m2 = make_float2(-2.0f, -2.0f);
#pragma unroll
      for (int A = 0; A < ND; ++A) {
        float wv[V];
        if (!WSRC) Pack<V>::ldcg(w + A * plane, e, wv);  // border faces store 0
#pragma unroll
        for (int hh = 0; hh < H; ++hh) {
          float2 a, b, c;
          face_forms2<V, ND>(wf, wg, A, hh, a, b, c);
          if (WSRC) {
            const bool in = pos[A] < lim[A];
            wv[2 * hh] = in ? (tp.weights_mode == 1 ? 1.0f : edge_weight(a.x, nis2[2 * hh])) : 0.0f;
            wv[2 * hh + (V > 1)] = in ? (tp.weights_mode == 1 ? 1.0f : edge_weight(a.y, nis2[2 * hh + (V > 1)])) : 0.0f;
          }
          fa[A][hh] = __fadd2_rn(a, eps22);
          fb[A][hh] = __fmul2_rn(m2, b);
          fc[A][hh] = c;
          wA2[A][hh] = make_float2(todo[2 * hh] ? wv[2 * hh] : 0.0f, todo[2 * hh + (V > 1)] ? wv[2 * hh + (V > 1)] : 0.0f);
        }
      }
#pragma unroll
      for (int q = 0; q < TV_KA; ++q) {
        const float t = tp.t[min(k0 + q, CTR_MAX_ARMIJO - 1)];
        const float2 t2 = make_float2(t, t);
#pragma unroll
        for (int hh = 0; hh < H; ++hh) {
          float2 acc2 = make_float2(0.0f, 0.0f);
#pragma unroll
          for (int A = 0; A < ND; ++A) {
            float2 rad = __ffma2_rn(t2, __ffma2_rn(t2, fc[A][hh], fb[A][hh]), fa[A][hh]);
            rad.x = fmaxf(rad.x, 1e-30f); rad.y = fmaxf(rad.y, 1e-30f);
            acc2 = __ffma2_rn(__fmul2_rn(wA2[A][hh], rad), make_float2(rsqrt_fast(rad.x), rsqrt_fast(rad.y)), acc2);
          }
          et[q * V + 2 * hh] += acc2.x;
          et[q * V + 2 * hh + (V > 1)] += acc2.y;
        }
      }
#pragma unroll
      for (int hh = 0; hh < H; ++hh) {
        float2 ws = make_float2(0.0f, 0.0f);
#pragma unroll
        for (int A = 0; A < ND; ++A) ws = __fadd2_rn(ws, wA2[A][hh]);
#pragma unroll
        for (int q = 0; q < TV_KA; ++q) {
          et[q * V + 2 * hh] = fmaf(-eps, ws.x, et[q * V + 2 * hh]);
          et[q * V + 2 * hh + (V > 1)] = fmaf(-eps, ws.y, et[q * V + 2 * hh + (V > 1)]);
        }
      }
    } else {
    // phase 1: the three forms of every face (the windows die here), eps^2 folded into a
      float fa[ND][V], fb[ND][V], fc[ND][V], wA[ND][V];
  #pragma unroll
      for (int A = 0; A < ND; ++A) {
        if (!WSRC) Pack<V>::ldcg(w + A * plane, e, wA[A]);  // border faces store 0
  #pragma unroll
        for (int s = 0; s < V; ++s) {
          float a, b, c;
          face_forms<V, ND>(wf, wg, A, s, a, b, c);
          if (WSRC) wA[A][s] = pos[A] < lim[A] ? (tp.weights_mode == 1 ? 1.0f : edge_weight(a, nis2[s])) : 0.0f;
          fa[A][s] = a + eps2;
          fb[A][s] = -2.0f * b;
          fc[A][s] = c;
          if (!todo[s]) wA[A][s] = 0.0f;
        }
      }
      // phase 2: sum_A w_A sqrt(N0^2(t_q) + eps^2) per candidate; the "- eps sum w" part does not depend on t
  #pragma unroll
      for (int q = 0; q < TV_KA; ++q) {
        const float t = tp.t[min(k0 + q, CTR_MAX_ARMIJO - 1)];
  #pragma unroll
        for (int A = 0; A < ND; ++A)
  #pragma unroll
          for (int s = 0; s < V; ++s) {
            const float rad = fmaxf(fmaf(t, fmaf(t, fc[A][s], fb[A][s]), fa[A][s]), 1e-30f);
            et[q * V + s] = fmaf(wA[A][s] * rad, rsqrt_fast(rad), et[q * V + s]);
          }
      }
      {
        float wsumv[V];
  #pragma unroll
        for (int s = 0; s < V; ++s) {
          wsumv[s] = 0.0f;
  #pragma unroll
          for (int A = 0; A < ND; ++A) wsumv[s] += wA[A][s];
  #pragma unroll
          for (int q = 0; q < TV_KA; ++q) et[q * V + s] = fmaf(-eps, wsumv[s], et[q * V + s]);
        }
      }
    }
    }
  }  // rr
  // block reduction. TV energies: fp32 column sums over the 32 lanes of a warp through shared memory (32
  // values per round, transposed so that lane q adds value q of all lanes in lane order), then fp64.
#pragma unroll
  for (int r0 = 0; r0 < NE; r0 += 32) {
#pragma unroll
    for (int q = 0; q < 32; ++q)
      if (r0 + q < NE) colsum[wid][q][lane] = et[r0 + q];
    __syncwarp();
    if (r0 + lane < NE) {
      float sum = 0.0f;
#pragma unroll 8
      for (int l = 0; l < 32; ++l) sum += colsum[wid][lane][l];
      wsum[wid][r0 + lane] = (double)sum;
    }
    __syncwarp();
  }
#pragma unroll
  for (int q = 0; q < 3 * V; ++q) {
    const double t = warp_sum(dd[q]);
    if (lane == 0) wsum[wid][NE + q] = t;
  }
  __syncthreads();
  if (tid < NV) {
    double t = 0.0;
#pragma unroll
    for (int ww = 0; ww < TV_TW; ++ww) t += wsum[ww][tid];
    part[((size_t)g * nblk + blk) * NV + tid] = t;
  }
}

// one block per slice group: adds the block partials in a fixed order, assembles E(t_k) in fp64 and takes
// the Armijo decision (reading S14/S25) for each slice of the group
template <int V>
__global__ void __launch_bounds__(1024) k_tv_trial_finish(const double* __restrict__ part, int nblk, TvParams tp, int k0,
                                                          int ndim, Scal sc) {
  constexpr int NE = TV_KA * V, NV = NE + 3 * V, ROWS = 1024 / NV;
  __shared__ double sm[ROWS][NV];
  __shared__ double tot[NV];
  const int g = blockIdx.x, t = threadIdx.x;
  const int n = t % NV, row = t / NV;
  bool any = false;
#pragma unroll
  for (int s = 0; s < V; ++s) any |= sc.kacc[g * V + s] < 0;
  if (!any) return;  // k_tv_trial wrote nothing for this group
  if (row < ROWS) {
    double acc = 0.0;
    const double* p = part + (size_t)g * nblk * NV + n;
#pragma unroll 4
    for (int b = row; b < nblk; b += ROWS) acc += __ldcg(p + (size_t)b * NV);
    sm[row][n] = acc;
  }
  __syncthreads();
  if (t < NV) {
    double acc = 0.0;
    for (int r = 0; r < ROWS; ++r) acc += sm[r][t];
    tot[t] = acc;
  }
  __syncthreads();
  if (t < V) {
    const int sl = g * V + t;
    if (sc.kacc[sl] < 0) {
      const double e0 = sc.e0[sl], g2 = sc.g2[sl];
      const double D0 = tot[NE + t], D1 = tot[NE + V + t], D2 = tot[NE + 2 * V + t];
      for (int q = 0; q < TV_KA && k0 + q < tp.kmax; ++q) {
        const double tk = (double)tp.t[k0 + q];
        const double E = 0.5 * (double)tp.lambda * (D0 - 2.0 * tk * D1 + tk * tk * D2) + tot[q * V + t] / (double)ndim;
        if (E <= e0 - (double)tp.c_armijo * tk * g2) {
          sc.kacc[sl] = k0 + q;
          sc.tacc[sl] = tp.t[k0 + q];
          break;
        }
      }
    }
  }
}

// a6.2 + a7  f <- f - t g for slices that accepted a step; optional positivity clamp; sweep record.
template <int V>
__global__ void __launch_bounds__(256) k_tv_apply(Dims d, float* __restrict__ f, const float* __restrict__ gin, Scal sc,
                                                  int clamp, StatRing ring) {
  const int g = blockIdx.y;
  const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
  if (blockIdx.x == 0 && g == 0) {
    // the sweep record of every slice, then the sweep counter moves on (one block: no other block reads it)
    ctr_sweep_stat* rec = ring.slot();
    for (int sl = threadIdx.x; sl < ring.Bp; sl += 256) {
      rec[sl].e0 = sc.e0[sl];
      rec[sl].g2 = sc.g2[sl];
      rec[sl].k = sc.kacc[sl];
    }
    __syncthreads();
    if (threadIdx.x == 0) *ring.sweep = *ring.sweep + 1ull;
  }
  if (idx >= (size_t)d.npix) return;
  const size_t e = (size_t)g * d.npix + idx;
  float fv[V], gv[V];
  Pack<V>::ldcg(f, e, fv);
  Pack<V>::ldcg(gin, e, gv);
#pragma unroll
  for (int s = 0; s < V; ++s) {
    const float t = sc.tacc[g * V + s];  // 0 when nothing was accepted
    float nf = sc.kacc[g * V + s] >= 0 ? fmaf(-t, gv[s], fv[s]) : fv[s];
    if (clamp) nf = fmaxf(nf, 0.0f);
    fv[s] = nf;
  }
  Pack<V>::st(f, e, fv);
}

template <int V>
__global__ void __launch_bounds__(256) k_clamp(Dims d, float* __restrict__ f) {
  const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
  if (idx >= (size_t)d.npix) return;
  const size_t e = (size_t)blockIdx.y * d.npix + idx;
  float fv[V];
  Pack<V>::ldcg(f, e, fv);
#pragma unroll
  for (int s = 0; s < V; ++s) fv[s] = fmaxf(fv[s], 0.0f);
  Pack<V>::st(f, e, fv);
}

// ---------------------------------------------------------------------------------------------
// host drivers
// ---------------------------------------------------------------------------------------------
static StatRing stat_slot(ctr_handle* h) {
  StatRing r;
  r.base = h->stats;
  r.sweep = h->d_sweep;
  r.Bp = h->d.G * h->d.V;
  return r;
}

// weight planes for the caller (ctr_update_weights, and the last sweep of ctr_reconstruct_w): magnitudes to
// h->n0, three radix passes over them, w = exp(-N0^2/sigma^2)
template <int V, int ND>
static int tv_update_weights_t(ctr_handle* h, const float* f, float* w, cudaStream_t st) {
  const Dims& d = h->d;
  const int rows = tv_rows(d, 4, TV_MAXROWS(d, 8), 148 * 16);
  const dim3 grid = vox_grid(d, rows), block(32, 4);
  const int Bp = d.G * d.V;
  const float eps2 = h->p.eps * h->p.eps;
  const StatRing rec = stat_slot(h);
  ProfScope prof(h, CTR_PROF_TV, st);
  k_tv_faces<V, ND><<<grid, block, 0, st>>>(d, rows, f, h->n0, h->hist);
  CTR_LAUNCHED(h);
  if (h->p.weights_mode == 1) {
    // plain TV: weights are 1, sigma is not needed (the record says 0)
    CTR_CUDA(h, cudaMemsetAsync(h->hist, 0, sizeof(unsigned) * 2048 * Bp, st));
  } else {
    k_tv_select<<<Bp, 256, 0, st>>>(h->sc, h->hist, 2048, 20, 1, 0, h->sel_k, eps2, rec, 0, 0u);
    CTR_LAUNCHED(h);
    k_tv_hist<V, ND><<<grid, block, 0, st>>>(d, rows, h->n0, h->hist, h->sc, 10, 1023u, 20);
    CTR_LAUNCHED(h);
    k_tv_select<<<Bp, 256, 0, st>>>(h->sc, h->hist, 1024, 10, 0, 0, 0, eps2, rec, 0, 0u);
    CTR_LAUNCHED(h);
    k_tv_hist<V, ND><<<grid, block, 0, st>>>(d, rows, h->n0, h->hist, h->sc, 0, 1023u, 10);
    CTR_LAUNCHED(h);
    k_tv_select<<<Bp, 256, 0, st>>>(h->sc, h->hist, 1024, 0, 0, 1, 0, eps2, rec, 0, 0u);
    CTR_LAUNCHED(h);
  }
  k_tv_weights<V, ND><<<grid, block, 0, st>>>(d, rows, h->n0, w, h->sc, h->p.weights_mode, rec);
  CTR_LAUNCHED(h);
  return CTR_OK;
}

int tv_update_weights(ctr_handle* h, const float* f, float* w, cudaStream_t st) {
  if (h->d.ndim == 3) return tv_update_weights_t<1, 3>(h, f, w, st);
  return h->d.V == 1 ? tv_update_weights_t<1, 2>(h, f, w, st) : tv_update_weights_t<4, 2>(h, f, w, st);
}

static TvParams make_tv_params(const ctr_handle* h, float lambda) {
  TvParams tp;
  tp.lambda = lambda;
  tp.eps = h->p.eps;
  tp.c_armijo = h->p.armijo_c;
  tp.kmax = h->p.armijo_max;
  tp.weights_mode = h->p.weights_mode;
  double t = (double)h->p.armijo_t0;
  for (int k = 0; k < CTR_MAX_ARMIJO; ++k) {
    tp.t[k] = (float)t;
    t *= (double)h->p.armijo_rho;
  }
  return tp;
}

// gradient + Armijo trials + update; WSRC = 0: weights from the planes w, WSRC = 1: weights on the fly from
// sc.sigma2 (fused path)
template <int V, int ND, int WSRC>
static int tv_descend_t(ctr_handle* h, float* f, const float* v, const float* w, float lambda, int clamp, cudaStream_t st) {
  const Dims& d = h->d;
  const int rows = tv_rows(d, 4, TV_MAXROWS(d, 8), 148 * 16);
  const dim3 grid = vox_grid(d, rows), block(32, 4);
  const TvParams tp = make_tv_params(h, lambda);
  float* g = h->gimg;
  k_tv_gradient<V, ND, WSRC><<<grid, block, 0, st>>>(d, rows, f, v, w, g, tp, h->sc, h->part, h->counters + 2 * d.G, stat_slot(h));
  CTR_LAUNCHED(h);
  const int trows = tv_rows(d, TV_TW, TV_MAXROWS(d, 16), 148 * 8);
  const dim3 tgrid((d.nx + 31) / 32, ((d.ny + TV_TW * trows - 1) / (TV_TW * trows)) * d.nz, d.G), tblock(32, TV_TW);
  for (int k0 = 0; k0 < tp.kmax; k0 += TV_KA) {
    k_tv_trial<V, ND, WSRC><<<tgrid, tblock, 0, st>>>(d, trows, f, g, v, w, tp, k0, h->sc, h->part);
    CTR_LAUNCHED(h);
    k_tv_trial_finish<V><<<d.G, 1024, 0, st>>>(h->part, (int)(tgrid.x * tgrid.y), tp, k0, d.ndim, h->sc);
    CTR_LAUNCHED(h);
  }
  k_tv_apply<V><<<dim3((d.npix + 255) / 256, d.G), 256, 0, st>>>(d, f, g, h->sc, clamp, stat_slot(h));
  CTR_LAUNCHED(h);
  h->sweep_count++;
  return CTR_OK;
}

int tv_sweep(ctr_handle* h, float* f, const float* v, const float* w, float lambda, int clamp, cudaStream_t st) {
  ProfScope prof(h, CTR_PROF_TV, st);
  if (h->d.ndim == 3) return tv_descend_t<1, 3, 0>(h, f, v, w, lambda, clamp, st);
  return h->d.V == 1 ? tv_descend_t<1, 2, 0>(h, f, v, w, lambda, clamp, st) : tv_descend_t<4, 2, 0>(h, f, v, w, lambda, clamp, st);
}

// One GD sweep of ctr_reconstruct without any plane: sigma by the fused selection (k_tv_scan1 / k_tv_scan23 above),
// then gradient, trials and update with the weights evaluated on the fly.
template <int V, int ND>
static int tv_sweep_fused_t(ctr_handle* h, float* f, const float* v, float lambda, int clamp, int pos, cudaStream_t st) {
  const Dims& d = h->d;
  ProfScope prof(h, CTR_PROF_TV, st);
  if (h->p.weights_mode == 0) {
    const int rows = tv_rows(d, 8, TV_MAXROWS(d, 8), 148 * 8);
    const dim3 grid = vox_grid(d, rows, 8), block(32, 8);
    const int Bp = d.G * d.V;
    const float eps2 = h->p.eps * h->p.eps;
    const StatRing rec = stat_slot(h);
    // large problems: the fast first pass, and the full one only for the groups in which a slice missed
    const bool fast = TV_FAST_SCAN && h->nimg * sizeof(float) >= ((size_t)32 << 20);
    if (fast) {
      k_tv_scan1f<V, ND><<<grid, block, 0, st>>>(d, rows, f, h->hist, h->sc, h->cand, h->cand_cap);
      CTR_LAUNCHED(h);
      k_tv_select_f<<<(Bp + 127) / 128, 128, 0, st>>>(h->sc, h->hist, Bp, h->sel_k, h->cand_cap);
      CTR_LAUNCHED(h);
    }
    k_tv_scan1<V, ND><<<grid, block, 0, st>>>(d, rows, f, h->hist, h->sc, h->cand, h->cand_cap, fast ? 1 : 0);
    CTR_LAUNCHED(h);
    k_tv_select<<<Bp, 256, 0, st>>>(h->sc, h->hist, 2048, 20, 1, 0, h->sel_k, eps2, rec, 1, h->cand_cap, 0, fast ? V : 0);
    CTR_LAUNCHED(h);
    k_tv_scan23<V, ND><<<grid, block, 0, st>>>(d, rows, f, h->hist, h->sc, h->cand, h->cand_cap, 10, 1023u, 20);
    CTR_LAUNCHED(h);
    k_tv_select<<<Bp, 256, 0, st>>>(h->sc, h->hist, 1024, 10, 0, 0, 0, eps2, rec, 1, h->cand_cap);
    CTR_LAUNCHED(h);
    k_tv_scan23<V, ND><<<grid, block, 0, st>>>(d, rows, f, h->hist, h->sc, h->cand, h->cand_cap, 0, 1023u, 10);
    CTR_LAUNCHED(h);
    k_tv_select<<<Bp, 256, 0, st>>>(h->sc, h->hist, 1024, 0, 0, 1, 0, eps2, rec, 1, h->cand_cap, pos);
    CTR_LAUNCHED(h);
  }
  return tv_descend_t<V, ND, 1>(h, f, v, nullptr, lambda, clamp, st);
}

int tv_sweep_fused(ctr_handle* h, float* f, const float* v, float lambda, int clamp, int pos, cudaStream_t st) {
  if (h->d.ndim == 3) return tv_sweep_fused_t<1, 3>(h, f, v, lambda, clamp, pos, st);
  return h->d.V == 1 ? tv_sweep_fused_t<1, 2>(h, f, v, lambda, clamp, pos, st) : tv_sweep_fused_t<4, 2>(h, f, v, lambda, clamp, pos, st);
}

int tv_clamp(ctr_handle* h, float* f, cudaStream_t st) {
  const Dims& d = h->d;
  dim3 grid((d.npix + 255) / 256, d.G);
  if (d.V == 1) k_clamp<1><<<grid, 256, 0, st>>>(d, f);
  else k_clamp<4><<<grid, 256, 0, st>>>(d, f);
  CTR_LAUNCHED(h);
  return CTR_OK;
}

}  // namespace ctr
