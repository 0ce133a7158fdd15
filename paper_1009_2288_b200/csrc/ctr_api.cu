// C ABI of libctr (include/ctr.h): handle management, layout conversion, CGLS and the outer loop.
#include <math.h>
#include <stdlib.h>

#include <new>

#include "ctr_common.cuh"
#include "ctr_internal.h"

using namespace ctr;

namespace ctr {

// ---------------------------------------------------------------------------------------------
// ABI <-> internal layout. ABI: [B][n] floats. Internal (V = 4): [G][n] float4, lane c = slice 4g+c,
// missing slices are zero. V = 1 uses the ABI arrays in place (no copies).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_pack4(const float* __restrict__ src, float* __restrict__ dst, size_t n, int B) {
  const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
  const int g = blockIdx.y, pl = blockIdx.z, G = gridDim.y;
  if (idx >= n) return;
  float o[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const int sl = 4 * g + c;
    o[c] = sl < B ? __ldg(src + ((size_t)pl * B + sl) * n + idx) : 0.0f;
  }
  reinterpret_cast<float4*>(dst)[((size_t)pl * G + g) * n + idx] = make_float4(o[0], o[1], o[2], o[3]);
}

__global__ void __launch_bounds__(256) k_unpack4(const float* __restrict__ src, float* __restrict__ dst, size_t n, int B) {
  const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
  const int g = blockIdx.y, pl = blockIdx.z, G = gridDim.y;
  if (idx >= n) return;
  const float4 t = __ldg(reinterpret_cast<const float4*>(src) + ((size_t)pl * G + g) * n + idx);
  const float o[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const int sl = 4 * g + c;
    if (sl < B) dst[((size_t)pl * B + sl) * n + idx] = o[c];
  }
}

static int pack(ctr_handle* h, const float* src, float* dst, size_t n, int planes, cudaStream_t st) {
  dim3 grid((unsigned)((n + 255) / 256), h->d.G, planes);
  ProfScope prof(h, CTR_PROF_LAYOUT, st);
  k_pack4<<<grid, 256, 0, st>>>(src, dst, n, h->d.B);
  CTR_LAUNCHED(h);
  return CTR_OK;
}
static int unpack(ctr_handle* h, const float* src, float* dst, size_t n, int planes, cudaStream_t st) {
  dim3 grid((unsigned)((n + 255) / 256), h->d.G, planes);
  ProfScope prof(h, CTR_PROF_LAYOUT, st);
  k_unpack4<<<grid, 256, 0, st>>>(src, dst, n, h->d.B);
  CTR_LAUNCHED(h);
  return CTR_OK;
}

// ---------------------------------------------------------------------------------------------
// a3  CGLS vector updates (App. I steps 2, 3, 5), per-slice scalars from device.
// The arrays are [GS][nl] V-packs with nl = n * LQ: pack idx of super-group gs belongs to slice group
// gs * LQ + idx % LQ (slice-interleaved layout; LQ = 1, V = 1 for a single slice).
// ---------------------------------------------------------------------------------------------
template <int V>
__global__ void __launch_bounds__(256) k_sino_axpy(size_t nl, int LQ, float* __restrict__ r, const float* __restrict__ q,
                                                   Scal sc) {
  const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
  const int gs = blockIdx.y;
  if (idx >= nl) return;
  const int sl0 = (gs * LQ + (int)(idx % LQ)) * V;
  float rv[V], qv[V];
  Pack<V>::ldcg(r, (size_t)gs * nl + idx, rv);
  Pack<V>::ldcg(q, (size_t)gs * nl + idx, qv);
#pragma unroll
  for (int c = 0; c < V; ++c) rv[c] = fmaf(-sc.a[sl0 + c], qv[c], rv[c]);  // r <- r - a P s
  Pack<V>::st(r, (size_t)gs * nl + idx, rv);
}

// s <- g + beta s (App. I step 5, :435; first = 1: s <- g) and store the unit gradient g/||g||
// as the next basis vector of the re-orthogonalisation (S24).
template <int V>
__global__ void __launch_bounds__(256) k_img_supdate(size_t nl, int LQ, float* __restrict__ s, const float* __restrict__ gi,
                                                     float* __restrict__ bnew, Scal sc, int first) {
  const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
  const int gs = blockIdx.y;
  if (idx >= nl) return;
  const int sl0 = (gs * LQ + (int)(idx % LQ)) * V;
  float sv[V], gv[V], bv[V];
  Pack<V>::ldcg(gi, (size_t)gs * nl + idx, gv);
  if (first) {
#pragma unroll
    for (int c = 0; c < V; ++c) sv[c] = gv[c];
  } else {
    Pack<V>::ldcg(s, (size_t)gs * nl + idx, sv);
#pragma unroll
    for (int c = 0; c < V; ++c) sv[c] = fmaf(sc.beta[sl0 + c], sv[c], gv[c]);
  }
  Pack<V>::st(s, (size_t)gs * nl + idx, sv);
  if (bnew) {
#pragma unroll
    for (int c = 0; c < V; ++c) bv[c] = gv[c] * sc.ginv[sl0 + c];
    Pack<V>::st(bnew, (size_t)gs * nl + idx, bv);
  }
}

template <int V>
__global__ void __launch_bounds__(256) k_img_uupdate(size_t nl, int LQ, float* __restrict__ u, const float* __restrict__ s,
                                                     Scal sc) {
  const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
  const int gs = blockIdx.y;
  if (idx >= nl) return;
  const int sl0 = (gs * LQ + (int)(idx % LQ)) * V;
  float uv[V], sv[V];
  Pack<V>::ldcg(u, (size_t)gs * nl + idx, uv);
  Pack<V>::ldcg(s, (size_t)gs * nl + idx, sv);
#pragma unroll
  for (int c = 0; c < V; ++c) uv[c] = fmaf(sc.a[sl0 + c], sv[c], uv[c]);  // u <- u + a s
  Pack<V>::st(u, (size_t)gs * nl + idx, uv);
}

// Re-orthogonalisation of the CGLS gradients (S24). In exact arithmetic P^T r^(m+1) is
// orthogonal to every earlier P^T r^(i) (Hestenes & Stiefel); in fp32 that is lost
// after ~6 iterations and the iterate then lags the exact one by a whole step. What is lost is the
// orthogonality to the FIRST gradients (the dominant singular directions converge first): projecting
// g against b_0..b_3 only tracks the oracle's full re-orthogonalisation to 1e-6 on every config
// (S24, table), at a constant cost per iteration. Classical Gram-Schmidt against them:
//   pass 1 (k_reorth_dots): c_i = <b_i, g> for NB basis vectors per launch (per-thread fp32 partial
//                           sums over a thread's elements, everything above that in fp64)
//   pass 2 (k_reorth_sub) : g <- g - sum_i c_i b_i, gamma' = ||g||^2, beta = gamma'/gamma (:432)
#define REORTH_NB 4   /* basis vectors per k_reorth_dots launch (= CTR_MAX_BASIS: one launch) */
static_assert(CTR_MAX_BASIS >= 1 && CTR_MAX_BASIS <= REORTH_NB,
              "CTR_MAX_BASIS must be 1..4: k_reorth_dots / k_finish handle REORTH_NB = 4 basis vectors per launch");
template <int V>
__global__ void __launch_bounds__(256) k_reorth_dots(size_t nl, int LQ, size_t nimg, const float* __restrict__ gi,
                                                     const float* __restrict__ basis, int i0, int nb, int Bp, Scal sc,
                                                     double* part, unsigned* counter) {
  const int gs = blockIdx.y;
  float acc[(REORTH_NB + 1) * V];  // slots [q][c]: <b_q, g> for q < NB, ||g||^2 for q = NB
#pragma unroll
  for (int q = 0; q < (REORTH_NB + 1) * V; ++q) acc[q] = 0.0f;
  // grid-stride loop (the stride is a multiple of 256, hence of LQ: a thread stays in its segment)
#pragma unroll 2
  for (size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x; idx < nl; idx += (size_t)gridDim.x * 256) {
    {
      float gv[V];
      Pack<V>::ldcg(gi, (size_t)gs * nl + idx, gv);
#pragma unroll
      for (int c = 0; c < V; ++c) acc[REORTH_NB * V + c] = fmaf(gv[c], gv[c], acc[REORTH_NB * V + c]);
#pragma unroll
      for (int q = 0; q < REORTH_NB; ++q) {
        if (q < nb) {
          float bv[V];
          Pack<V>::ldcg(basis + (size_t)(i0 + q) * nimg, (size_t)gs * nl + idx, bv);
#pragma unroll
          for (int c = 0; c < V; ++c) acc[q * V + c] = fmaf(bv[c], gv[c], acc[q * V + c]);
        }
      }
    }
  }
  double red[(REORTH_NB + 1) * V];
#pragma unroll
  for (int q = 0; q < (REORTH_NB + 1) * V; ++q) red[q] = (double)acc[q];
  block_partials_q<(REORTH_NB + 1) * V, 8>(red, LQ, part + (size_t)gs * gridDim.x * LQ * (REORTH_NB + 1) * V, blockIdx.x, threadIdx.x);
}

// g' = g - sum_i c_i b_i (never stored), s <- g' + beta s (App. I step 5, :435; first = 1: s <- g') and the
// next unit gradient b_new = g'/||g'||, in one pass. gamma' = ||g'||^2 comes from Pythagoras in k_finish
// (||g||^2 - sum c_i^2: the b_i are orthonormal), so no separate subtraction pass is needed.
template <int V>
__global__ void __launch_bounds__(256) k_img_update(size_t nl, int LQ, size_t nimg, const float* __restrict__ gi,
                                                    const float* __restrict__ basis, int nb, int Bp, float* __restrict__ s,
                                                    float* __restrict__ bnew, int first, Scal sc) {
  const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
  const int gs = blockIdx.y;
  if (idx >= nl) return;
  const int sl0 = (gs * LQ + (int)(idx % LQ)) * V;
  const size_t e = (size_t)gs * nl + idx;
  float gv[V], sv[V];
  Pack<V>::ldcg(gi, e, gv);
#pragma unroll 4
  for (int q = 0; q < nb; ++q) {
    float bv[V];
    Pack<V>::ldcg(basis + (size_t)q * nimg, e, bv);
#pragma unroll
    for (int c = 0; c < V; ++c) gv[c] = fmaf(-sc.coef[(size_t)q * Bp + sl0 + c], bv[c], gv[c]);
  }
  if (first) {
#pragma unroll
    for (int c = 0; c < V; ++c) sv[c] = gv[c];
  } else {
    Pack<V>::ldcg(s, e, sv);
#pragma unroll
    for (int c = 0; c < V; ++c) sv[c] = fmaf(sc.beta[sl0 + c], sv[c], gv[c]);
  }
  Pack<V>::st(s, e, sv);
  if (bnew) {
#pragma unroll
    for (int c = 0; c < V; ++c) gv[c] *= sc.ginv[sl0 + c];
    Pack<V>::st(bnew, e, gv);
  }
}

// Finishing pass of the segmented reductions: block (q, gs) adds the partials part[gs][b][q][0..N) over the
// blocks b in a fixed order and applies the scalar update of the producing kernel:
//   FIN_ALPHA  N = V:       delta = ||P s||^2 -> a = gamma/delta            (App. I step 1)
//   FIN_COEF   N = (NB+1) V: c_i = <b_i, g> (S24) and gamma' = ||g||^2 - sum_i c_i^2 = ||g - sum c_i b_i||^2,
//                            beta = gamma'/gamma, 1/sqrt(gamma')               (App. I step 4, :432)
template <int N>
__global__ void __launch_bounds__(1024) k_finish(int mode, const double* __restrict__ part, int nblk, int LQ, int V,
                                                int i0, int nb, int Bp, int first, Scal sc) {
  __shared__ double sm[1024];
  __shared__ double tot[N];
  const int q = blockIdx.x, gs = blockIdx.y, t = threadIdx.x;
  const int n = t % N, b0 = t / N;
  constexpr int NB0 = 1024 / N;  // block rows: 1024 threads keep the chain of dependent loads short
  double acc = 0.0;
  const double* p = part + ((size_t)gs * nblk * LQ + q) * N + n;
  if (b0 < NB0) {
#pragma unroll 4
    for (int b = b0; b < nblk; b += NB0) acc += __ldcg(p + (size_t)b * LQ * N);
  }
  sm[t] = acc;
  __syncthreads();
  double sum = 0.0;
  if (t < N) {
    for (int j = 0; j < NB0; ++j) sum += sm[j * N + n];
    tot[t] = sum;
  }
  __syncthreads();
  if (t >= N) return;
  const int c = n % V, sl = (gs * LQ + q) * V + c;
  if (mode == CTR_FIN_ALPHA) {
    const double gamma = sc.gamma[sl];
    const float a = (sum > 0.0 && gamma > 0.0) ? (float)(gamma / sum) : 0.0f;  // S4
    sc.a[sl] = a;
    // lazy phase: u_hat += a s_hat leaves out a sum_i e_i b_i; remember it per slice (nb = coefficients in use)
    for (int i = 0; i < nb; ++i) sc.dco[(size_t)i * Bp + sl] = fmaf(a, sc.eco[(size_t)i * Bp + sl], sc.dco[(size_t)i * Bp + sl]);
  } else {
    const int qb = n / V, NBV = N / V - 1;
    if (qb < nb) sc.coef[(size_t)(i0 + qb) * Bp + sl] = (float)sum;
    if (qb == NBV) {
      // the coefficients are applied in fp32: use their rounded values in Pythagoras too
      double g2 = sum;
      for (int i = 0; i < nb; ++i) { const double ci = (double)(float)tot[i * V + c]; g2 -= ci * ci; }
      if (g2 < 0.0) g2 = 0.0;
      if (!first) {
        const double gamma = sc.gamma[sl];
        sc.beta[sl] = gamma > 0.0 ? (float)(g2 / gamma) : 0.0f;  // S4
      }
      sc.gamma[sl] = g2;
      sc.ginv[sl] = g2 > 0.0 ? (float)(1.0 / sqrt(g2)) : 0.0f;
    }
  }
}

int reduce_finish(ctr_handle* h, int mode, int N, int nblk, int i0, int nb, int first, cudaStream_t st) {
  const Dims& d = h->d;
  dim3 grid(d.LQ, d.GS);
  const int Bp = d.G * d.V;
  switch (N) {
    case 1: k_finish<1><<<grid, 1024, 0, st>>>(mode, h->part, nblk, d.LQ, d.V, i0, nb, Bp, first, h->sc); break;
    case 4: k_finish<4><<<grid, 1024, 0, st>>>(mode, h->part, nblk, d.LQ, d.V, i0, nb, Bp, first, h->sc); break;
    case 5: k_finish<5><<<grid, 1024, 0, st>>>(mode, h->part, nblk, d.LQ, d.V, i0, nb, Bp, first, h->sc); break;
    default: k_finish<20><<<grid, 1024, 0, st>>>(mode, h->part, nblk, d.LQ, d.V, i0, nb, Bp, first, h->sc); break;
  }
  CTR_LAUNCHED(h);
  return CTR_OK;
}


// ---------------------------------------------------------------------------------------------
// Lazy phase of the re-orthogonalised CGLS (S24, section 5). Once the CTR_MAX_BASIS unit gradients b_i
// exist, projecting every new gradient against them in image space costs two passes over 4 image-size vectors
// per iteration (most of the CGLS vector traffic at 64 slices). Both passes move to the sinogram side, which is
// 5 x smaller:
//   c_i = <b_i, P^T r> = <P b_i, r>, and P b_i comes for free: s_i = g'_i + beta_i s_(i-1) gives
//         P b_i = (q_i - beta_i q_(i-1)) / ||g'_i|| from the q = P s that CGLS forms anyway;
//   the projected direction is never materialised: the kernels carry s_hat = g + beta s_hat (the recurrence as
//         printed) and per-slice coefficients e_i <- c_i + beta e_i with s = s_hat - sum_i e_i b_i, hence
//         q = P s = P s_hat - sum_i e_i P b_i (sinogram side), and u = u_hat - sum_i d_i b_i with d_i += a e_i is
//         materialised once, after the last iteration.
// In exact arithmetic this is the iteration of vec_direction() term for term; in fp32 it tracks the oracle as
// closely (tests/test_oracle_pins.py emulates both).
// ---------------------------------------------------------------------------------------------
#ifndef CTR_LAZY_BLOCKS
#define CTR_LAZY_BLOCKS 592 /* grid cap of the lazy-phase reduction kernels, 4 blocks per SM: their partials are finished by k_finish* (c4 vector work 1.85 / 1.82 / 2.11 ms for 1184 / 592 / 296) */
#endif
#ifndef CTR_LAZY_V1
#define CTR_LAZY_V1 4
#endif
static_assert(CTR_LAZY_BLOCKS <= CTR_REDUCE_BLOCKS && CTR_LAZY_V1 <= 16, "part2 is sized for CTR_REDUCE_BLOCKS blocks x 16 segments");
// explicit phase, iteration m < CTR_MAX_BASIS: P b_m = (q - beta q_prev) / ||g'_m|| (first: q / ||g'_0||); q_prev <- q
template <int V>
__global__ void __launch_bounds__(256) k_sino_pb(size_t nl, int LQ, const float* __restrict__ q, float* __restrict__ qprev,
                                                 float* __restrict__ pbm, int first, Scal sc) {
  const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
  const int gs = blockIdx.y;
  if (idx >= nl) return;
  const int sl0 = (gs * LQ + (int)(idx % LQ)) * V;
  const size_t e = (size_t)gs * nl + idx;
  float qv[V], pv[V], o[V];
  Pack<V>::ldcg(q, e, qv);
  if (!first) Pack<V>::ldcg(qprev, e, pv);
#pragma unroll
  for (int c = 0; c < V; ++c) o[c] = (first ? qv[c] : fmaf(-sc.beta[sl0 + c], pv[c], qv[c])) * sc.ginv[sl0 + c];
  Pack<V>::st(pbm, e, o);
  Pack<V>::st(qprev, e, qv);
}

// lazy phase: q <- q_hat - sum_i e_i P b_i, and delta = ||q||^2 (block partials, N = V)
template <int V>
__global__ void __launch_bounds__(256) k_sino_correct(size_t nl, int LQ, size_t nsino, float* __restrict__ q,
                                                      const float* __restrict__ pb, int nb, int Bp, Scal sc, double* part) {
  const int gs = blockIdx.y;
  float acc[V];
#pragma unroll
  for (int c = 0; c < V; ++c) acc[c] = 0.0f;
  for (size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x; idx < nl; idx += (size_t)gridDim.x * 256) {
    const int sl0 = (gs * LQ + (int)(idx % LQ)) * V;
    const size_t e = (size_t)gs * nl + idx;
    float qv[V];
    Pack<V>::ldcg(q, e, qv);
#pragma unroll 4
    for (int i = 0; i < nb; ++i) {
      float pv[V];
      Pack<V>::ldcg(pb + (size_t)i * nsino, e, pv);
#pragma unroll
      for (int c = 0; c < V; ++c) qv[c] = fmaf(-sc.eco[(size_t)i * Bp + sl0 + c], pv[c], qv[c]);
    }
    Pack<V>::st(q, e, qv);
#pragma unroll
    for (int c = 0; c < V; ++c) acc[c] = fmaf(qv[c], qv[c], acc[c]);
  }
  double red[V];
#pragma unroll
  for (int c = 0; c < V; ++c) red[c] = (double)acc[c];
  block_partials_q<V, 8>(red, LQ, part + (size_t)gs * gridDim.x * LQ * V, blockIdx.x, threadIdx.x);
}

// lazy phase: r <- r - a q (App. I step 3, :429) and c_i = <P b_i, r> for the new r (block partials, N = REORTH_NB V)
template <int V>
__global__ void __launch_bounds__(256) k_sino_axpy_dots(size_t nl, int LQ, size_t nsino, float* __restrict__ r,
                                                        const float* __restrict__ q, const float* __restrict__ pb, int nb,
                                                        Scal sc, double* part) {
  const int gs = blockIdx.y;
  float acc[REORTH_NB * V];
#pragma unroll
  for (int t = 0; t < REORTH_NB * V; ++t) acc[t] = 0.0f;
  for (size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x; idx < nl; idx += (size_t)gridDim.x * 256) {
    const int sl0 = (gs * LQ + (int)(idx % LQ)) * V;
    const size_t e = (size_t)gs * nl + idx;
    float rv[V], qv[V];
    Pack<V>::ldcg(r, e, rv);
    Pack<V>::ldcg(q, e, qv);
#pragma unroll
    for (int c = 0; c < V; ++c) rv[c] = fmaf(-sc.a[sl0 + c], qv[c], rv[c]);
    Pack<V>::st(r, e, rv);
#pragma unroll
    for (int i = 0; i < REORTH_NB; ++i) {
      if (i < nb) {
        float pv[V];
        Pack<V>::ldcg(pb + (size_t)i * nsino, e, pv);
#pragma unroll
        for (int c = 0; c < V; ++c) acc[i * V + c] = fmaf(pv[c], rv[c], acc[i * V + c]);
      }
    }
  }
  double red[REORTH_NB * V];
#pragma unroll
  for (int t = 0; t < REORTH_NB * V; ++t) red[t] = (double)acc[t];
  block_partials_q<REORTH_NB * V, 8>(red, LQ, part + (size_t)gs * gridDim.x * LQ * REORTH_NB * V, blockIdx.x, threadIdx.x);
}

// lazy phase: ||g||^2 per slice (block partials, N = V). k_reorth_dots with nb = 0 would do, but its grid is sized for
// five streams per thread (two blocks per SM): 25 us for the 64-MiB gradient against 12 us here.
template <int V>
__global__ void __launch_bounds__(256) k_img_norm(size_t nl, int LQ, const float* __restrict__ gi, double* part) {
  const int gs = blockIdx.y;
  float acc[V];
#pragma unroll
  for (int c = 0; c < V; ++c) acc[c] = 0.0f;
#pragma unroll 4
  for (size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x; idx < nl; idx += (size_t)gridDim.x * 256) {
    float gv[V];
    Pack<V>::ldcg(gi, (size_t)gs * nl + idx, gv);
#pragma unroll
    for (int c = 0; c < V; ++c) acc[c] = fmaf(gv[c], gv[c], acc[c]);
  }
  double red[V];
#pragma unroll
  for (int c = 0; c < V; ++c) red[c] = (double)acc[c];
  block_partials_q<V, 8>(red, LQ, part + (size_t)gs * gridDim.x * LQ * V, blockIdx.x, threadIdx.x);
}

// lazy phase, scalar step after P^T: block (q, gs) sums ||g||^2 and the c_i (partials of k_sino_axpy_dots), then gamma' = ||g||^2 - sum c_i^2, beta = gamma'/gamma
// (:432) and e_i <- c_i + beta e_i
template <int V>
__global__ void __launch_bounds__(1024) k_finish_lazy(const double* __restrict__ part, int nblk, int N1, int off1,
                                                     const double* __restrict__ part2, int nblk2, int LQ, int nb, int Bp,
                                                     Scal sc) {
  // ||g||^2: value off1 + c of the N1 values per (block, segment) in `part` (k_img_norm: N1 = V, off1 = 0)
  constexpr int N2 = REORTH_NB * V, NT = V + N2;  // values wanted: ||g||^2 [V], c [NB][V]
  constexpr int ROWS = 1024 / NT;
  __shared__ double sm[ROWS][NT];
  __shared__ double tot[NT];
  const int q = blockIdx.x, gs = blockIdx.y, t = threadIdx.x;
  const int n = t % NT, row = t / NT;
  if (row < ROWS) {
    double acc = 0.0;
    if (n < V) {
      const double* p = part + ((size_t)gs * nblk * LQ + q) * N1 + off1 + n;
#pragma unroll 4
      for (int b = row; b < nblk; b += ROWS) acc += __ldcg(p + (size_t)b * LQ * N1);
    } else {
      const double* p = part2 + ((size_t)gs * nblk2 * LQ + q) * N2 + (n - V);
#pragma unroll 4
      for (int b = row; b < nblk2; b += ROWS) acc += __ldcg(p + (size_t)b * LQ * N2);
    }
    sm[row][n] = acc;
  }
  __syncthreads();
  if (t < NT) {
    double acc = 0.0;
    for (int r = 0; r < ROWS; ++r) acc += sm[r][t];
    tot[t] = acc;
  }
  __syncthreads();
  if (t >= V) return;
  const int sl = (gs * LQ + q) * V + t;
  double g2 = tot[t];
  float cf[REORTH_NB];
#pragma unroll
  for (int i = 0; i < REORTH_NB; ++i) {
    cf[i] = i < nb ? (float)tot[V + i * V + t] : 0.0f;
    g2 -= (double)cf[i] * (double)cf[i];  // the coefficients act in fp32: Pythagoras with their rounded values
  }
  if (g2 < 0.0) g2 = 0.0;
  const double gamma = sc.gamma[sl];
  const float beta = gamma > 0.0 ? (float)(g2 / gamma) : 0.0f;  // S4
  sc.beta[sl] = beta;
  sc.gamma[sl] = g2;
  sc.ginv[sl] = g2 > 0.0 ? (float)(1.0 / sqrt(g2)) : 0.0f;
#pragma unroll
  for (int i = 0; i < REORTH_NB; ++i)
    if (i < nb) {
      sc.coef[(size_t)i * Bp + sl] = cf[i];
      sc.eco[(size_t)i * Bp + sl] = fmaf(beta, sc.eco[(size_t)i * Bp + sl], cf[i]);
    }
}

// after the last iteration: u <- u_hat - sum_i d_i b_i
template <int V>
__global__ void __launch_bounds__(256) k_img_fixup(size_t nl, int LQ, size_t nimg, float* __restrict__ u,
                                                   const float* __restrict__ basis, int nb, int Bp, Scal sc) {
  const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
  const int gs = blockIdx.y;
  if (idx >= nl) return;
  const int sl0 = (gs * LQ + (int)(idx % LQ)) * V;
  const size_t e = (size_t)gs * nl + idx;
  float uv[V];
  Pack<V>::ldcg(u, e, uv);
#pragma unroll 4
  for (int i = 0; i < nb; ++i) {
    float bv[V];
    Pack<V>::ldcg(basis + (size_t)i * nimg, e, bv);
#pragma unroll
    for (int c = 0; c < V; ++c) uv[c] = fmaf(-sc.dco[(size_t)i * Bp + sl0 + c], bv[c], uv[c]);
  }
  Pack<V>::st(u, e, uv);
}

static int vec_sino_axpy(ctr_handle* h, float* r, const float* q, cudaStream_t st) {
  const Dims& d = h->d;
  const size_t nl = (size_t)d.nray * d.LQ;
  dim3 grid((unsigned)((nl + 255) / 256), d.GS);
  ProfScope prof(h, CTR_PROF_VECTOR, st);
  if (d.V == 1) k_sino_axpy<1><<<grid, 256, 0, st>>>(nl, d.LQ, r, q, h->sc);
  else k_sino_axpy<4><<<grid, 256, 0, st>>>(nl, d.LQ, r, q, h->sc);
  CTR_LAUNCHED(h);
  return CTR_OK;
}
// u <- u + tau g with one step for all slices: the (P1) update of Eq. 8, any layout
__global__ void __launch_bounds__(256) k_axpy_const(size_t n4, float4* __restrict__ u, const float4* __restrict__ g, float tau) {
  const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
  if (idx >= n4) return;
  float4 uv = __ldcg(u + idx);
  const float4 gv = __ldcg(g + idx);
  uv.x = fmaf(tau, gv.x, uv.x); uv.y = fmaf(tau, gv.y, uv.y); uv.z = fmaf(tau, gv.z, uv.z); uv.w = fmaf(tau, gv.w, uv.w);
  u[idx] = uv;
}
__global__ void __launch_bounds__(256) k_axpy_const1(size_t n, float* __restrict__ u, const float* __restrict__ g, float tau) {
  const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
  if (idx < n) u[idx] = fmaf(tau, __ldcg(g + idx), u[idx]);
}

static int vec_img_uupdate(ctr_handle* h, float* u, const float* s, cudaStream_t st) {
  const Dims& d = h->d;
  const size_t nl = (size_t)d.npix * d.LQ;
  dim3 grid((unsigned)((nl + 255) / 256), d.GS);
  ProfScope prof(h, CTR_PROF_VECTOR, st);
  if (d.V == 1) k_img_uupdate<1><<<grid, 256, 0, st>>>(nl, d.LQ, u, s, h->sc);
  else k_img_uupdate<4><<<grid, 256, 0, st>>>(nl, d.LQ, u, s, h->sc);
  CTR_LAUNCHED(h);
  return CTR_OK;
}
// App. I steps 4-5 with the re-orthogonalisation of S24: c_i = <b_i, g>, gamma' = ||g - sum c_i b_i||^2,
// beta = gamma'/gamma; then s <- g' + beta s and the next unit gradient, without ever storing g'
static int vec_direction(ctr_handle* h, const float* g, int nb, int first, float* bnew, cudaStream_t st) {
  const Dims& d = h->d;
  const size_t nl = (size_t)d.npix * d.LQ;
  const int Bp = d.G * d.V;
  const unsigned want = (unsigned)((nl + 255) / 256);
  unsigned dcap = (unsigned)(h->dots_blocks / d.GS);
  if (dcap < 1) dcap = 1;
  dim3 grid(want, d.GS);
  dim3 dgrid(want < dcap ? want : dcap, d.GS);  // exactly one resident wave of the register-heavy kernel
  ProfScope prof(h, CTR_PROF_VECTOR, st);
  if (nb > CTR_MAX_BASIS) nb = CTR_MAX_BASIS;
  if (d.V == 1) k_reorth_dots<1><<<dgrid, 256, 0, st>>>(nl, d.LQ, h->nimg, g, h->basis, 0, nb, Bp, h->sc, h->part, h->counters + 4 * d.G);
  else k_reorth_dots<4><<<dgrid, 256, 0, st>>>(nl, d.LQ, h->nimg, g, h->basis, 0, nb, Bp, h->sc, h->part, h->counters + 4 * d.G);
  CTR_LAUNCHED(h);
  int rc = reduce_finish(h, CTR_FIN_COEF, (REORTH_NB + 1) * d.V, (int)dgrid.x, 0, nb, first, st);
  if (rc) return rc;
  if (d.V == 1) k_img_update<1><<<grid, 256, 0, st>>>(nl, d.LQ, h->nimg, g, h->basis, nb, Bp, h->s, bnew, first, h->sc);
  else k_img_update<4><<<grid, 256, 0, st>>>(nl, d.LQ, h->nimg, g, h->basis, nb, Bp, h->s, bnew, first, h->sc);
  CTR_LAUNCHED(h);
  return CTR_OK;
}

// lazy phase helpers (kernels above)
static int vec_sino_pb(ctr_handle* h, int m, cudaStream_t st) {
  const Dims& d = h->d;
  const size_t nl = (size_t)d.nray * d.LQ;
  dim3 grid((unsigned)((nl + 255) / 256), d.GS);
  ProfScope prof(h, CTR_PROF_VECTOR, st);
  float* pbm = h->pbasis + (size_t)m * h->nsino;
  if (d.V == 1) k_sino_pb<1><<<grid, 256, 0, st>>>(nl, d.LQ, h->q, h->qprev, pbm, m == 0, h->sc);
  else k_sino_pb<4><<<grid, 256, 0, st>>>(nl, d.LQ, h->q, h->qprev, pbm, m == 0, h->sc);
  CTR_LAUNCHED(h);
  return CTR_OK;
}
static dim3 sino_reduce_grid(const ctr_handle* h) {
  const Dims& d = h->d;
  const size_t nl = (size_t)d.nray * d.LQ;
  const unsigned want = (unsigned)((nl + 255) / 256);
  // (a single problem loads 4 bytes per thread and stream where a batch loads 16: four times the blocks in flight)
  unsigned cap = (unsigned)(CTR_LAZY_BLOCKS * (d.V == 1 ? CTR_LAZY_V1 : 1) / d.GS);
  if (cap < 1) cap = 1;
  return dim3(want < cap ? want : cap, d.GS);
}
// q <- q_hat - sum e_i P b_i, a = gamma/||q||^2, d_i += a e_i
static int vec_sino_correct(ctr_handle* h, cudaStream_t st) {
  const Dims& d = h->d;
  const size_t nl = (size_t)d.nray * d.LQ;
  const dim3 grid = sino_reduce_grid(h);
  const int Bp = d.G * d.V;
  ProfScope prof(h, CTR_PROF_VECTOR, st);
  if (d.V == 1) k_sino_correct<1><<<grid, 256, 0, st>>>(nl, d.LQ, h->nsino, h->q, h->pbasis, CTR_MAX_BASIS, Bp, h->sc, h->part);
  else k_sino_correct<4><<<grid, 256, 0, st>>>(nl, d.LQ, h->nsino, h->q, h->pbasis, CTR_MAX_BASIS, Bp, h->sc, h->part);
  CTR_LAUNCHED(h);
  return reduce_finish(h, CTR_FIN_ALPHA, d.V, (int)grid.x, 0, CTR_MAX_BASIS, 0, st);
}
// r <- r - a q and the partials of c_i = <P b_i, r>; returns the block count of the partials in *nblk2
static int vec_sino_axpy_dots(ctr_handle* h, int* nblk2, cudaStream_t st) {
  const Dims& d = h->d;
  const size_t nl = (size_t)d.nray * d.LQ;
  const dim3 grid = sino_reduce_grid(h);
  ProfScope prof(h, CTR_PROF_VECTOR, st);
  if (d.V == 1) k_sino_axpy_dots<1><<<grid, 256, 0, st>>>(nl, d.LQ, h->nsino, h->r, h->q, h->pbasis, CTR_MAX_BASIS, h->sc, h->part2);
  else k_sino_axpy_dots<4><<<grid, 256, 0, st>>>(nl, d.LQ, h->nsino, h->r, h->q, h->pbasis, CTR_MAX_BASIS, h->sc, h->part2);
  CTR_LAUNCHED(h);
  *nblk2 = (int)grid.x;
  return CTR_OK;
}
// ||g||^2, then gamma', beta, e_i, then s_hat <- g + beta s_hat
static int vec_direction_lazy(ctr_handle* h, const float* g, int nblk2, cudaStream_t st) {
  const Dims& d = h->d;
  const size_t nl = (size_t)d.npix * d.LQ;
  const int Bp = d.G * d.V;
  const unsigned want = (unsigned)((nl + 255) / 256);
  unsigned ncap = (unsigned)(CTR_LAZY_BLOCKS * (d.V == 1 ? CTR_LAZY_V1 : 1) / d.GS);
  if (ncap < 1) ncap = 1;
  dim3 grid(want, d.GS), ngrid(want < ncap ? want : ncap, d.GS), fgrid(d.LQ, d.GS);
  ProfScope prof(h, CTR_PROF_VECTOR, st);
  if (d.V == 1) {
    k_img_norm<1><<<ngrid, 256, 0, st>>>(nl, d.LQ, g, h->part);
    CTR_LAUNCHED(h);
    k_finish_lazy<1><<<fgrid, 1024, 0, st>>>(h->part, (int)ngrid.x, 1, 0, h->part2, nblk2, d.LQ, CTR_MAX_BASIS, Bp, h->sc);
    CTR_LAUNCHED(h);
    k_img_supdate<1><<<grid, 256, 0, st>>>(nl, d.LQ, h->s, g, nullptr, h->sc, 0);
  } else {
    k_img_norm<4><<<ngrid, 256, 0, st>>>(nl, d.LQ, g, h->part);
    CTR_LAUNCHED(h);
    k_finish_lazy<4><<<fgrid, 1024, 0, st>>>(h->part, (int)ngrid.x, 4, 0, h->part2, nblk2, d.LQ, CTR_MAX_BASIS, Bp, h->sc);
    CTR_LAUNCHED(h);
    k_img_supdate<4><<<grid, 256, 0, st>>>(nl, d.LQ, h->s, g, nullptr, h->sc, 0);
  }
  CTR_LAUNCHED(h);
  return CTR_OK;
}
static int vec_img_fixup(ctr_handle* h, float* u, cudaStream_t st) {
  const Dims& d = h->d;
  const size_t nl = (size_t)d.npix * d.LQ;
  dim3 grid((unsigned)((nl + 255) / 256), d.GS);
  ProfScope prof(h, CTR_PROF_VECTOR, st);
  if (d.V == 1) k_img_fixup<1><<<grid, 256, 0, st>>>(nl, d.LQ, h->nimg, u, h->basis, CTR_MAX_BASIS, d.G * d.V, h->sc);
  else k_img_fixup<4><<<grid, 256, 0, st>>>(nl, d.LQ, h->nimg, u, h->basis, CTR_MAX_BASIS, d.G * d.V, h->sc);
  CTR_LAUNCHED(h);
  return CTR_OK;
}

static int op_forward(ctr_handle* h, const float* img, float* out, int mode, const float* bs, cudaStream_t st) {
  return h->d.ndim == 3 ? cone_forward(h, img, out, mode, bs, st) : fan_forward(h, img, out, mode, bs, st);
}
static int op_back(ctr_handle* h, const float* sino, float* out, int mode, const float* s, float* u, cudaStream_t st) {
  return h->d.ndim == 3 ? cone_back(h, sino, out, mode, s, u, st) : fan_back(h, sino, out, mode, s, u, st);
}

// NEXT-1 inside the solvers (ctr_params.backprojector = 1): out = B sino with B the paper's pixel-driven Eq. (11)
// in place of the exact transpose. k_back_eq11 works on the ABI layouts, so a batch goes
// SI -> ABI -> Eq. (11) -> SI through h->q and h->n0, which are free whenever a backprojection is due.
static int op_back_eq11(ctr_handle* h, const float* sino, float* out, cudaStream_t st) {
  if (h->d.V == 1) return fan_back_eq11(h, sino, out, st);
  int rc;
  if ((rc = si_to_abi(h, sino, h->q, h->d.nray, st))) return rc;
  if ((rc = fan_back_eq11(h, h->q, h->n0, st))) return rc;
  return si_from_abi(h, h->n0, out, h->d.npix, st);
}

// CGLS on internal-layout arrays (gradients re-orthogonalised, S24). u: in x0 /
// out u^(M). The last iteration only needs u (its P^T r and s are never used, O4), so it ends with a
// plain u += a s. With the unmatched pair (backprojector = 1) the "gradients" B r are not orthogonal even in
// exact arithmetic: the recurrence runs as printed, nothing is projected out.
static int cgls_internal(ctr_handle* h, const float* b, float* u, int n_iter, bool x0_zero, cudaStream_t st) {
  if (n_iter <= 0) return CTR_OK;
  int rc;
  const bool eq11 = h->p.backprojector == 1;
  if (x0_zero) {
    CTR_CUDA(h, cudaMemcpyAsync(h->r, b, h->nsino * sizeof(float), cudaMemcpyDeviceToDevice, st));  // r0 = y
  } else if ((rc = op_forward(h, u, h->r, 1, b, st))) return rc;                                    // r0 = y - P u0
  if ((rc = eq11 ? op_back_eq11(h, h->r, h->gimg, st) : op_back(h, h->r, h->gimg, 0, nullptr, nullptr, st))) return rc;  // g0 = P^T r0
  if ((rc = vec_direction(h, h->gimg, 0, 1, eq11 ? nullptr : h->basis, st))) return rc;             // gamma0, s0 = g0, b_0
  // lazy phase (see k_sino_pb ...): from iteration CTR_MAX_BASIS on, if the solve is long enough to get there
  // (only where the image-size vectors stream from HBM: for a single slice everything is L2-resident and the extra
  // launches cost more than the traffic they save - c3: 1.93 -> 2.00 ms per outer iteration, measured)
  const bool lazy = !eq11 && !(h->g.flags & CTR_GEOM_NO_LAZY_CGLS) && n_iter > CTR_MAX_BASIS + 1 &&
                    h->nimg * sizeof(float) >= ((size_t)32 << 20);
  // (Folding the sinogram-side correction into k_si_forward_tab's epilogue and ||g||^2 into k_si_back_quad's was built
  // and measured at c4: forward +0.21, back +0.14, vector -0.26 ms per step - a net loss of 0.1 ms against the
  // separate 12-15 us passes used here: a block-wide reduction at the end of a projector block costs as much.)
  if (lazy) {
    const size_t nco = sizeof(float) * (size_t)h->d.G * h->d.V * CTR_MAX_BASIS;
    CTR_CUDA(h, cudaMemsetAsync(h->sc.eco, 0, nco, st));
    CTR_CUDA(h, cudaMemsetAsync(h->sc.dco, 0, nco, st));
  }
  for (int m = 0; m < n_iter; ++m) {
    if (lazy && m >= CTR_MAX_BASIS) {
      if ((rc = op_forward(h, h->s, h->q, 0, nullptr, st))) return rc;   // q_hat = P s_hat
      if ((rc = vec_sino_correct(h, st))) return rc;                     // q = P s, a = gamma/||q||^2, d += a e
      if (m == n_iter - 1) {
        if ((rc = vec_img_uupdate(h, u, h->s, st))) return rc;           // u_hat += a s_hat
        return vec_img_fixup(h, u, st);                                  // u = u_hat - sum d_i b_i
      }
      int nblk2 = 0;
      if ((rc = vec_sino_axpy_dots(h, &nblk2, st))) return rc;           // r -= a q, c_i = <P b_i, r>
      if ((rc = op_back(h, h->r, h->gimg, 2, h->s, u, st))) return rc;   // g = P^T r, u_hat += a s_hat
      if ((rc = vec_direction_lazy(h, h->gimg, nblk2, st))) return rc;   // ||g||^2, gamma', beta, e_i, s_hat = g + beta s_hat
      continue;
    }
    if ((rc = op_forward(h, h->s, h->q, 2, nullptr, st))) return rc;     // q = P s, a = gamma/||q||^2
    if (m == n_iter - 1) return vec_img_uupdate(h, u, h->s, st);         // u += a s
    if (lazy && (rc = vec_sino_pb(h, m, st))) return rc;                 // P b_m from q_m and q_(m-1)
    if (lazy && m == CTR_MAX_BASIS - 1) {
      // the gradient of the next iteration is the first one projected on the sinogram side
      int nblk2 = 0;
      if ((rc = vec_sino_axpy_dots(h, &nblk2, st))) return rc;
      if ((rc = op_back(h, h->r, h->gimg, 2, h->s, u, st))) return rc;
      if ((rc = vec_direction_lazy(h, h->gimg, nblk2, st))) return rc;
      continue;
    }
    if ((rc = vec_sino_axpy(h, h->r, h->q, st))) return rc;              // r -= a q
    if (eq11) {
      if ((rc = vec_img_uupdate(h, u, h->s, st))) return rc;             // u += a s
      if ((rc = op_back_eq11(h, h->r, h->gimg, st))) return rc;          // g = B r
      if ((rc = vec_direction(h, h->gimg, 0, 0, nullptr, st))) return rc;  // gamma', beta, s = g + beta s
      continue;
    }
    if ((rc = op_back(h, h->r, h->gimg, 2, h->s, u, st))) return rc;     // g = P^T r, u += a s
    float* bnew = (m + 1 < CTR_MAX_BASIS) ? h->basis + (size_t)(m + 1) * h->nimg : nullptr;
    if ((rc = vec_direction(h, h->gimg, m + 1, 0, bnew, st))) return rc;  // g' _|_ b_0.., gamma', beta, s = g' + beta s, b_{m+1}
  }
  return CTR_OK;
}

// (P1) of Eq. 8 (NEXT-4): n plain gradient updates u <- u - tau P^T (P u - y) on internal-layout arrays
static int p1_internal(ctr_handle* h, const float* b, float* u, int n, float tau, cudaStream_t st) {
  int rc;
  const bool eq11 = h->p.backprojector == 1;
  for (int m = 0; m < n; ++m) {
    if ((rc = op_forward(h, u, h->r, 1, b, st))) return rc;                                          // r = y - P u
    if ((rc = eq11 ? op_back_eq11(h, h->r, h->gimg, st) : op_back(h, h->r, h->gimg, 0, nullptr, nullptr, st))) return rc;
    ProfScope prof(h, CTR_PROF_VECTOR, st);
    if (h->d.V == 1) k_axpy_const1<<<(unsigned)((h->nimg + 255) / 256), 256, 0, st>>>(h->nimg, u, h->gimg, tau);
    else k_axpy_const<<<(unsigned)((h->nimg / 4 + 255) / 256), 256, 0, st>>>(h->nimg / 4, (float4*)u, (const float4*)h->gimg, tau);
    CTR_LAUNCHED(h);
  }
  return CTR_OK;
}

// double -> float copy for ctr_update_weights' optional sigma output
__global__ void k_d2f(const double* __restrict__ s, float* __restrict__ o, int n) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) o[i] = (float)s[i];
}

static bool aligned16(const void* p) { return p && (((uintptr_t)p) & 15u) == 0; }

static int check_params(const ctr_params* p) {
  if (!p) return CTR_EINVAL;
  if (p->n_outer < 0 || p->n_cgls < 0 || p->n_gd < 0) return CTR_EINVAL;
  if (!(p->lambda >= 0.0f) || !(p->sigma_quantile > 0.0f && p->sigma_quantile <= 1.0f)) return CTR_EINVAL;
  if (!(p->eps >= 0.0f) || !(p->armijo_t0 > 0.0f) || !(p->armijo_rho > 0.0f && p->armijo_rho < 1.0f)) return CTR_EINVAL;
  if (!(p->armijo_c >= 0.0f) || p->armijo_max < 1 || p->armijo_max > CTR_MAX_ARMIJO) return CTR_EINVAL;
  if (p->weights_mode != 0 && p->weights_mode != 1) return CTR_EINVAL;
  if (p->fidelity_mode != 0 && p->fidelity_mode != 1) return CTR_EINVAL;
  if (p->backprojector != 0 && p->backprojector != 1) return CTR_EINVAL;
  if (!(p->p1_step >= 0.0f)) return CTR_EINVAL;
  return CTR_OK;
}

static void set_quantile(ctr_handle* h, float q) {
  const Dims& d = h->d;
  // number of interior faces per slice / volume (O6)
  unsigned long long S = 0;
  S += (unsigned long long)(d.nx - 1) * d.ny * d.nz;
  S += (unsigned long long)d.nx * (d.ny - 1) * d.nz;
  if (d.ndim == 3) S += (unsigned long long)d.nx * d.ny * (d.nz - 1);
  double kk = ceil((double)q * (double)S);
  unsigned long long k = kk < 1.0 ? 1ull : (unsigned long long)kk;
  if (k > S) k = S;
  if (S == 0) k = 0;
  h->sel_k = k;
  h->sel_q = q;
}

}  // namespace ctr

// =============================================================================================
extern "C" {

void ctr_default_params(ctr_params* p) {
  if (!p) return;
  p->n_outer = 1; p->n_cgls = 10; p->n_gd = 5;
  p->lambda = 0.01f; p->sigma_quantile = 0.90f; p->eps = 1e-4f;
  p->armijo_t0 = 1e-3f; p->armijo_rho = 0.5f; p->armijo_c = 0.5f; p->armijo_max = 16;
  p->weights_mode = 0; p->positivity = 1; p->warm_start = 0;
  p->fidelity_mode = 0; p->p1_step = 0.0f; p->backprojector = 0;
}

const char* ctr_strerror(int status) {
  switch (status) {
    case CTR_OK: return "ok";
    case CTR_EINVAL: return "invalid argument";
    case CTR_EGEOM: return "invalid geometry (source or detector inside the image circle)";
    case CTR_ENOMEM: return "out of memory";
    case CTR_ECUDA: return "CUDA error";
    case CTR_EARCH: return "device is not sm_100 (B200)";
    case CTR_ETOOBIG: return "problem exceeds the fixed scratch of ctr_forward_noalloc (max 512 x 512 pixels, 65536 rays, 4096 views)";
    default: return "unknown status";
  }
}

const char* ctr_last_error(const ctr_handle* h) { return h ? h->err : ""; }
const char* ctr_path_info(const ctr_handle* h) { return h ? h->path_info : ""; }
long long ctr_launch_count(const ctr_handle* h) { return h ? h->launches : 0; }

void ctr_destroy(ctr_handle* h) {
  if (!h) return;
  cudaDeviceSynchronize();
  void* bufs[] = {h->rays, h->rays2, h->views, h->viewsd, h->ximg, h->bsino, h->r, h->q, h->s, h->gimg, h->v, h->w, h->n0,
                  h->part, h->part2, h->counters, h->hist, h->scal_block, h->stats, h->d_sweep, h->basis, h->pbasis, h->qprev, h->win, h->imgT, h->win2, h->usi, h->cand, h->rt_tab, h->rt_cnt, h->rt_off, h->qidx, h->qwts, h->qcnt, h->ell_p.tab, h->ell_p.cap, h->ell_p.off, h->ell_pt.tab, h->ell_pt.cap, h->ell_pt.off};
  for (void* b : bufs)
    if (b) cudaFree(b);
  if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
  if (h->gstream) cudaStreamDestroy(h->gstream);
  if (h->prof_ev) {
    for (int i = 0; i < 2 * CTR_PROF_MAX; ++i) cudaEventDestroy(h->prof_ev[i]);
    free(h->prof_ev);
    free(h->prof_kind);
  }
  free(h->g.angles ? (void*)h->g.angles : nullptr);
  delete h;
}

int ctr_create(const ctr_geometry* g, ctr_handle** out) {
  if (!out) return CTR_EINVAL;
  *out = nullptr;
  if (!g) return CTR_EINVAL;
  if (g->ndim != 2 && g->ndim != 3) return CTR_EINVAL;
  if (g->nx < 1 || g->ny < 1 || g->nz < 1 || g->nviews < 1 || g->nu < 1 || g->nv < 1 || g->batch < 1) return CTR_EINVAL;
  if (g->ndim == 2 && (g->nz != 1 || g->nv != 1)) return CTR_EINVAL;
  if (g->ndim == 3 && (g->batch != 1 || g->det_type != 0)) return CTR_EINVAL;
  if (!(g->dx > 0) || !(g->dy > 0) || !(g->du > 0) || !(g->dso > 0) || !(g->dsd > g->dso)) return CTR_EINVAL;
  if (g->ndim == 3 && (!(g->dz > 0) || !(g->dv > 0))) return CTR_EINVAL;
  if (g->det_type != 0 && g->det_type != 1) return CTR_EINVAL;
  if (g->flags & ~(CTR_GEOM_NO_TABLES | CTR_GEOM_NO_GRAPHS | CTR_GEOM_NO_STORED_P | CTR_GEOM_NO_LAZY_CGLS)) return CTR_EINVAL;
  if ((long long)g->nx * g->ny * g->nz >= (1ll << 31) || (long long)g->nviews * g->nu * g->nv >= (1ll << 31)) return CTR_EINVAL;
  // source and detector must lie outside the circle circumscribing the grid (plus one voxel)
  {
    double hx = fabs((double)g->cx) + 0.5 * g->nx * (double)g->dx + g->dx;
    double hy = fabs((double)g->cy) + 0.5 * g->ny * (double)g->dy + g->dy;
    double rad = sqrt(hx * hx + hy * hy);
    if (!(g->dso > rad) || !((double)g->dsd - g->dso > rad)) return CTR_EGEOM;
  }
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return CTR_ECUDA;
  if (prop.major != 10) return CTR_EARCH;

  ctr_handle* h = new (std::nothrow) ctr_handle();
  if (!h) return CTR_ENOMEM;
  memset(h, 0, sizeof(*h));
  h->g = *g;
  h->g.angles = nullptr;
  if (g->angles) {
    float* a = (float*)malloc(sizeof(float) * g->nviews);
    if (!a) { delete h; return CTR_ENOMEM; }
    memcpy(a, g->angles, sizeof(float) * g->nviews);
    h->g.angles = a;
  }
  h->device = dev;
  ctr_default_params(&h->p);

  Dims& d = h->d;
  d.ndim = g->ndim;
  d.nx = g->nx; d.ny = g->ny; d.nz = g->nz;
  d.nviews = g->nviews; d.nu = g->nu; d.nv = g->nv;
  d.c0x = g->nx / 2; d.c0y = g->ny / 2; d.c0z = g->nz / 2;
  d.npix = g->nx * g->ny * g->nz;
  d.nray = g->nviews * g->nu * g->nv;
  d.B = g->batch;
  d.V = g->batch > 1 ? 4 : 1;
  {
    // groups of V slices; batched: LQ groups (a power of two <= 16) form a super-group of the
    // slice-interleaved layout, and the group count is padded to a whole number of super-groups
    const int g0 = (g->batch + d.V - 1) / d.V;
    d.LQ = 1;
    if (d.V == 4) while (d.LQ < 16 && d.LQ < g0) d.LQ *= 2;
    d.GS = (g0 + d.LQ - 1) / d.LQ;
    d.G = d.GS * d.LQ;
  }
  d.nvp = (g->nviews + 15) / 16 * 16;
  d.dx = g->dx; d.dy = g->dy; d.dz = g->ndim == 3 ? g->dz : 1.0f;
  d.xlo = (float)((double)g->cx - g->nx * (double)g->dx / 2.0);
  d.ylo = (float)((double)g->cy - g->ny * (double)g->dy / 2.0);
  d.zlo = (float)((double)g->cz - g->nz * (double)d.dz / 2.0);
  d.dso = g->dso; d.dsd = g->dsd;
  d.inv_du = 1.0f / g->du;
  d.inv_dv = g->ndim == 3 ? 1.0f / g->dv : 1.0f;
  d.dvz = g->ndim == 3 ? g->dv / g->dz : 1.0f;
  d.boff_u = (float)((g->nu - 1) / 2.0 - (double)g->u_off);
  d.boff_v = (float)((g->nv - 1) / 2.0 - (double)g->v_off);
  d.rvox = 0.5f * sqrtf(d.dx * d.dx + d.dy * d.dy + (g->ndim == 3 ? d.dz * d.dz : 0.0f));
  d.det_type = g->det_type;

  const int Bp = d.G * d.V;
  h->nimg = (size_t)Bp * d.npix;
  h->nsino = (size_t)Bp * d.nray;
  const size_t fb = sizeof(float);
  cudaError_t e = cudaSuccess;
  auto A = [&](void** p, size_t bytes) {
    if (e == cudaSuccess) e = cudaMalloc(p, bytes ? bytes : 16);
  };
  A((void**)&h->rays, sizeof(float4) * (size_t)d.nviews * d.nu);
  if (d.ndim == 3) A((void**)&h->rays2, sizeof(float4) * (size_t)d.nviews * d.nu);
  A((void**)&h->views, sizeof(float2) * d.nviews);
  A((void**)&h->viewsd, sizeof(double2) * d.nviews);
  A((void**)&h->win, sizeof(unsigned short) * (size_t)d.nviews * d.nx * d.ny);
  if (d.V == 1) A((void**)&h->imgT, h->nimg * fb);
  else {
    A((void**)&h->win2, sizeof(unsigned short) * (size_t)d.npix * d.nvp);
    A((void**)&h->usi, h->nimg * fb);
  }
  A((void**)&h->ximg, h->nimg * fb);
  A((void**)&h->bsino, h->nsino * fb);
  A((void**)&h->r, h->nsino * fb);
  A((void**)&h->q, h->nsino * fb);
  A((void**)&h->s, h->nimg * fb);
  A((void**)&h->gimg, h->nimg * fb);
  A((void**)&h->v, h->nimg * fb);
  A((void**)&h->w, h->nimg * fb * d.ndim);
  A((void**)&h->n0, h->nimg * fb * d.ndim);
  A((void**)&h->basis, h->nimg * fb * CTR_MAX_BASIS);  // unit CGLS gradients b_0..b_3 (S24)
  A((void**)&h->pbasis, h->nsino * fb * CTR_MAX_BASIS);  // P b_i, and q of the previous iteration (lazy CGLS phase)
  A((void**)&h->qprev, h->nsino * fb);
  A((void**)&h->part2, sizeof(double) * (size_t)CTR_REDUCE_BLOCKS * 16 * REORTH_NB * 4);  // [GS][blocks <= cap/GS][LQ][NB V]
  // partial sums: the largest user is the TV trial kernel (TV_KC * V slots per block)
  {
    size_t nblk_tv = (size_t)((d.nx + 31) / 32) * ((d.ny + 3) / 4) * d.nz;
    size_t nblk_p = (size_t)(d.nray + 127) / 128;
    size_t nblk = nblk_tv > nblk_p ? nblk_tv : nblk_p;
    h->part_len = (size_t)d.G * nblk * 8 * d.V;
    // Armijo trial pass: [G][blocks of 32 x 8 voxels][16 V + 3 V]
    size_t need_t = (size_t)d.G * ((size_t)((d.nx + 31) / 32) * ((d.ny + 3) / 4) * d.nz) * 19 * d.V;  // >= 4 rows per block
    if (need_t > h->part_len) h->part_len = need_t;
    // segmented reductions of the CGLS kernels: [GS][blocks][LQ][N] with N <= 8 * V
    size_t nblk_f = ((size_t)d.nray + 8 * (32 / d.LQ) - 1) / (8 * (32 / d.LQ));
    size_t nblk_q = nblk_f > CTR_REDUCE_BLOCKS ? nblk_f : CTR_REDUCE_BLOCKS;
    size_t need_q = (size_t)d.GS * nblk_q * d.LQ * 8 * d.V;
    if (need_q > h->part_len) h->part_len = need_q;
    A((void**)&h->part, h->part_len * sizeof(double));
  }
  A((void**)&h->counters, sizeof(unsigned) * CTR_NCOUNTERS * d.G);
  A((void**)&h->hist, sizeof(unsigned) * 2048 * Bp);
  A((void**)&h->stats, sizeof(ctr_sweep_stat) * (size_t)CTR_STAT_SWEEPS * Bp);
  A((void**)&h->d_sweep, 16);
  const size_t scal_bytes = (size_t)Bp * (3 * sizeof(double) + (5 + 3 * CTR_MAX_BASIS) * sizeof(float) + 10 * sizeof(unsigned) + 16);
  {
    // candidate lists of the fused sigma selection: a quarter of the faces of a slice / volume each
    unsigned long long S = (unsigned long long)(d.nx - 1) * d.ny * d.nz + (unsigned long long)d.nx * (d.ny - 1) * d.nz;
    if (d.ndim == 3) S += (unsigned long long)d.nx * d.ny * (d.nz - 1);
    unsigned long long cap = S / 4 + 1024;
    if (cap > 0x7fffffffull) cap = 0x7fffffffull;
    h->cand_cap = (unsigned)cap;
    A((void**)&h->cand, sizeof(unsigned) * (size_t)Bp * h->cand_cap);
  }
  A(&h->scal_block, scal_bytes);
  if (e != cudaSuccess) {
    int rc = e == cudaErrorMemoryAllocation ? CTR_ENOMEM : CTR_ECUDA;
    cudaGetLastError();
    ctr_destroy(h);
    return rc;
  }
  cudaMemset(h->counters, 0, sizeof(unsigned) * CTR_NCOUNTERS * d.G);
  cudaMemset(h->hist, 0, sizeof(unsigned) * 2048 * Bp);
  cudaMemset(h->scal_block, 0, scal_bytes);
  cudaMemset(h->stats, 0, sizeof(ctr_sweep_stat) * (size_t)CTR_STAT_SWEEPS * Bp);
  cudaMemset(h->d_sweep, 0, 16);
  {
    char* p = (char*)h->scal_block;
    h->sc.gamma = (double*)p; p += sizeof(double) * Bp;
    h->sc.e0 = (double*)p; p += sizeof(double) * Bp;
    h->sc.g2 = (double*)p; p += sizeof(double) * Bp;
    h->sc.a = (float*)p; p += sizeof(float) * Bp;
    h->sc.beta = (float*)p; p += sizeof(float) * Bp;
    h->sc.sigma2 = (float*)p; p += sizeof(float) * Bp;
    h->sc.tacc = (float*)p; p += sizeof(float) * Bp;
    h->sc.kacc = (int*)p; p += sizeof(int) * Bp;
    h->sc.sel_prefix = (unsigned*)p; p += sizeof(unsigned) * Bp;
    h->sc.sel_rank = (unsigned*)p; p += sizeof(unsigned) * Bp;
    h->sc.ginv = (float*)p; p += sizeof(float) * Bp;
    h->sc.coef = (float*)p; p += sizeof(float) * Bp * CTR_MAX_BASIS;
    h->sc.eco = (float*)p; p += sizeof(float) * Bp * CTR_MAX_BASIS;
    h->sc.dco = (float*)p; p += sizeof(float) * Bp * CTR_MAX_BASIS;
    h->sc.pred = (int*)p; p += sizeof(int) * Bp;
    h->sc.cand_cnt = (unsigned*)p; p += sizeof(unsigned) * Bp;
    h->sc.ovf = (unsigned*)p; p += sizeof(unsigned) * Bp;
    h->sc.hit = (int*)p; p += sizeof(int) * Bp;
    h->sc.lastbin = (int*)p; p += sizeof(int) * Bp;
    h->sc.jump = (int*)p; p += sizeof(int) * Bp;
    h->sc.fhit = (int*)p;
    cudaMemset(h->sc.pred, 0x80, sizeof(int) * Bp);  // a large negative bin: no prediction yet
    cudaMemset(h->sc.lastbin, 0x80, sizeof(int) * Bp);
  }
  set_quantile(h, h->p.sigma_quantile);
  {
    int per_sm = 0;
    cudaError_t oe = d.V == 1 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_reorth_dots<1>, 256, 0)
                              : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_reorth_dots<4>, 256, 0);
    if (oe != cudaSuccess || per_sm < 1) { cudaGetLastError(); per_sm = 2; }
    h->dots_blocks = per_sm * prop.multiProcessorCount;
    if (h->dots_blocks > CTR_REDUCE_BLOCKS) h->dots_blocks = CTR_REDUCE_BLOCKS;
  }
  if (cudaStreamCreateWithFlags(&h->gstream, cudaStreamNonBlocking) != cudaSuccess) {
    cudaGetLastError();
    h->gstream = nullptr;  // no capture stream: ctr_reconstruct launches kernel by kernel
  }
  int rc = d.ndim == 3 ? cone_build_tables(h) : fan_build_tables(h);
  if (rc == CTR_OK && d.ndim == 2 && d.V == 4) rc = si_build_hits(h);
  if (rc == CTR_OK && d.ndim == 2 && d.V == 4) rc = si_build_raytab(h);
  if (rc != CTR_OK) { ctr_destroy(h); return rc; }
  {
    // which kernels ctr_forward / ctr_back launch on this handle (the tables are built best effort)
    const char *fw, *bk;
    double table_mb = 0.0;
    if (d.V == 4) {
      fw = h->rt_tab ? "k_si_forward_tab" : "k_si_forward";
      bk = h->qwts ? "k_si_back_quad" : "k_si_back";
      table_mb = (double)h->rt_bytes / 1e6;
      if (h->qwts) table_mb += (double)((d.nx + 1) / 2) * ((d.ny + 1) / 2) * h->hits_cap * 20.0 / 1e6;
    } else {
      fw = h->ell_p.tab ? "k_ell_apply<P>" : (d.ndim == 3 ? "k_cone_forward" : "k_fan_forward");
      bk = h->ell_pt.tab ? "k_ell_apply<PT>" : (d.ndim == 3 ? "k_cone_back" : "k_fan_back");
      table_mb = (double)(h->ell_p.tab ? h->ell_p.bytes : 0) / 1e6 + (double)(h->ell_pt.tab ? h->ell_pt.bytes : 0) / 1e6;
    }
    snprintf(h->path_info, sizeof(h->path_info), "forward=%s;back=%s;tables_mb=%.1f;graphs=%d", fw, bk, table_mb,
             (h->gstream && !(g->flags & CTR_GEOM_NO_GRAPHS)) ? 1 : 0);
  }
  *out = h;
  return CTR_OK;
}

int ctr_set_params(ctr_handle* h, const ctr_params* p) {
  if (!h) return CTR_EINVAL;
  int rc = check_params(p);
  if (rc) return set_err(h, rc, "ctr_set_params: parameter out of range");
  if (p->backprojector == 1 && h->d.ndim != 2) return set_err(h, CTR_EINVAL, "ctr_set_params: Eq. (11) backprojector is 2D only");
  h->p = *p;
  set_quantile(h, p->sigma_quantile);
  return CTR_OK;
}

int ctr_forward(ctr_handle* h, const float* d_img, float* d_sino, void* stream) {
  if (!h) return CTR_EINVAL;
  if (!aligned16(d_img) || !aligned16(d_sino)) return set_err(h, CTR_EINVAL, "ctr_forward: NULL or misaligned pointer");
  cudaStream_t st = (cudaStream_t)stream;
  h->last_stream = st;
  if (h->d.V == 1) return op_forward(h, d_img, d_sino, 0, nullptr, st);
  int rc;
  if ((rc = si_from_abi(h, d_img, h->usi, h->d.npix, st))) return rc;
  if ((rc = op_forward(h, h->usi, h->q, 0, nullptr, st))) return rc;
  return si_to_abi(h, h->q, d_sino, h->d.nray, st);
}

int ctr_back(ctr_handle* h, const float* d_sino, float* d_img, void* stream) {
  if (!h) return CTR_EINVAL;
  if (!aligned16(d_img) || !aligned16(d_sino)) return set_err(h, CTR_EINVAL, "ctr_back: NULL or misaligned pointer");
  cudaStream_t st = (cudaStream_t)stream;
  h->last_stream = st;
  if (h->d.V == 1) return op_back(h, d_sino, d_img, 0, nullptr, nullptr, st);
  int rc;
  if ((rc = si_from_abi(h, d_sino, h->bsino, h->d.nray, st))) return rc;
  if ((rc = op_back(h, h->bsino, h->gimg, 0, nullptr, nullptr, st))) return rc;
  return si_to_abi(h, h->gimg, d_img, h->d.npix, st);
}

int ctr_back_pixel(ctr_handle* h, const float* d_sino, float* d_img, void* stream) {
  if (!h) return CTR_EINVAL;
  if (!aligned16(d_img) || !aligned16(d_sino)) return set_err(h, CTR_EINVAL, "ctr_back_pixel: NULL or misaligned pointer");
  if (h->d.ndim != 2) return set_err(h, CTR_EINVAL, "ctr_back_pixel: Eq. (11) is defined for 2D fan beams only");
  cudaStream_t st = (cudaStream_t)stream;
  h->last_stream = st;
  return fan_back_eq11(h, d_sino, d_img, st);
}

int ctr_cgls(ctr_handle* h, const float* d_b, float* d_x, int n_iter, void* stream) {
  if (!h) return CTR_EINVAL;
  if (!aligned16(d_b) || !aligned16(d_x)) return set_err(h, CTR_EINVAL, "ctr_cgls: NULL or misaligned pointer");
  if (n_iter < 0) return set_err(h, CTR_EINVAL, "ctr_cgls: n_iter < 0");
  if (n_iter == 0) return CTR_OK;
  cudaStream_t st = (cudaStream_t)stream;
  h->last_stream = st;
  if (h->d.V == 1) return cgls_internal(h, d_b, d_x, n_iter, false, st);
  int rc;
  if ((rc = si_from_abi(h, d_b, h->bsino, h->d.nray, st))) return rc;
  if ((rc = si_from_abi(h, d_x, h->usi, h->d.npix, st))) return rc;
  if ((rc = cgls_internal(h, h->bsino, h->usi, n_iter, false, st))) return rc;
  return si_to_abi(h, h->usi, d_x, h->d.npix, st);
}

int ctr_update_weights(ctr_handle* h, const float* d_x, float* d_w, float quantile, float* d_sigma, void* stream) {
  if (!h) return CTR_EINVAL;
  if (!aligned16(d_x) || !aligned16(d_w)) return set_err(h, CTR_EINVAL, "ctr_update_weights: NULL or misaligned pointer");
  if (!(quantile > 0.0f && quantile <= 1.0f)) return set_err(h, CTR_EINVAL, "ctr_update_weights: quantile not in (0,1]");
  cudaStream_t st = (cudaStream_t)stream;
  h->last_stream = st;
  const float q_saved = h->sel_q;
  set_quantile(h, quantile);
  int rc;
  if (h->d.V == 1) {
    rc = tv_update_weights(h, d_x, d_w, st);
  } else {
    rc = pack(h, d_x, h->ximg, h->d.npix, 1, st);
    if (!rc) rc = tv_update_weights(h, h->ximg, h->w, st);
    if (!rc) rc = unpack(h, h->w, d_w, h->d.npix, h->d.ndim, st);
  }
  set_quantile(h, q_saved);
  if (rc) return rc;
  if (d_sigma) {
    // sigma = sqrt(sigma^2) per true slice, from the sweep record just written
    const int Bp = h->d.G * h->d.V;
    ctr_sweep_stat* rec = h->stats + (size_t)(h->sweep_count % CTR_STAT_SWEEPS) * Bp;
    // strided device copy: sigma is the first double of each record
    CTR_CUDA(h, cudaMemcpy2DAsync(h->part, sizeof(double), rec, sizeof(ctr_sweep_stat), sizeof(double), h->d.B,
                                  cudaMemcpyDeviceToDevice, st));
    k_d2f<<<(h->d.B + 127) / 128, 128, 0, st>>>(h->part, d_sigma, h->d.B);
    CTR_LAUNCHED(h);
  }
  return CTR_OK;
}

int ctr_eptv_step(ctr_handle* h, float* d_x, const float* d_v, const float* d_w, float lambda, void* stream) {
  if (!h) return CTR_EINVAL;
  if (!aligned16(d_x) || !aligned16(d_v) || !aligned16(d_w))
    return set_err(h, CTR_EINVAL, "ctr_eptv_step: NULL or misaligned pointer");
  if (!(lambda >= 0.0f)) return set_err(h, CTR_EINVAL, "ctr_eptv_step: lambda < 0");
  cudaStream_t st = (cudaStream_t)stream;
  h->last_stream = st;
  if (h->d.V == 1) return tv_sweep(h, d_x, d_v, d_w, lambda, 0, st);
  int rc;
  if ((rc = pack(h, d_x, h->ximg, h->d.npix, 1, st))) return rc;
  if ((rc = pack(h, d_v, h->v, h->d.npix, 1, st))) return rc;
  if ((rc = pack(h, d_w, h->w, h->d.npix, h->d.ndim, st))) return rc;
  if ((rc = tv_sweep(h, h->ximg, h->v, h->w, lambda, 0, st))) return rc;
  return unpack(h, h->ximg, d_x, h->d.npix, 1, st);
}

int ctr_reconstruct_w(ctr_handle* h, const float* d_sino, float* d_img, float* d_w, const ctr_params* p, void* stream) {
  if (!h) return CTR_EINVAL;
  if (!aligned16(d_sino) || !aligned16(d_img) || (d_w && !aligned16(d_w)))
    return set_err(h, CTR_EINVAL, "ctr_reconstruct: NULL or misaligned pointer");
  int rc;
  if (p && (rc = ctr_set_params(h, p))) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  h->last_stream = st;
  h->sweep_count = 0;
  CTR_CUDA(h, cudaMemsetAsync(h->d_sweep, 0, sizeof(unsigned long long), st));
  const ctr_params& P = h->p;
  const bool direct = h->d.V == 1;
  float* f = direct ? d_img : h->ximg;
  const float* b = d_sino;
  if (!direct) {
    if ((rc = si_from_abi(h, d_sino, h->bsino, h->d.nray, st))) return rc;  // slice-interleaved
    b = h->bsino;
  }
  if (!P.warm_start) CTR_CUDA(h, cudaMemsetAsync(f, 0, h->nimg * sizeof(float), st));            // f^(0) = 0 (:171)
  else if (!direct && (rc = pack(h, d_img, h->ximg, h->d.npix, 1, st))) return rc;
  // one outer iteration (Steps 1-3 of the algorithm box), enqueued on stream s
  auto outer = [&](int it, bool x0_zero, bool want_w, cudaStream_t s_) -> int {
    int rc_;
    // Step 1 (:171): CGLS, or the (P1) gradient updates it replaced (fidelity_mode = 1)
    auto step1 = [&](float* u) -> int {
      return P.fidelity_mode == 1 ? p1_internal(h, b, u, P.n_cgls, P.p1_step, s_) : cgls_internal(h, b, u, P.n_cgls, x0_zero, s_);
    };
    if (direct) {
      if ((rc_ = step1(f))) return rc_;
    } else if (P.n_cgls > 0) {
      // batched: Step 1 runs in the slice-interleaved layout, the TV sweeps in the group-planar one
      if (x0_zero) CTR_CUDA(h, cudaMemsetAsync(h->usi, 0, h->nimg * sizeof(float), s_));
      else if ((rc_ = si_from_planar(h, f, h->usi, h->d.npix, s_))) return rc_;
      if ((rc_ = step1(h->usi))) return rc_;
      if ((rc_ = si_to_planar(h, h->usi, f, h->d.npix, s_))) return rc_;
    }
    if (P.n_gd > 0)
      CTR_CUDA(h, cudaMemcpyAsync(h->v, f, h->nimg * sizeof(float), cudaMemcpyDeviceToDevice, s_));  // v = CGLS result
    for (int sw = 0; sw < P.n_gd; ++sw) {                                                           // Step 2 (:172)
      const int clamp = (sw == P.n_gd - 1) && P.positivity;
      if (want_w && sw == P.n_gd - 1) {
        // the caller wants the weights of the last sweep: materialise them for this one sweep
        if ((rc_ = tv_update_weights(h, f, h->w, s_))) return rc_;
        if ((rc_ = tv_sweep(h, f, h->v, h->w, P.lambda, clamp, s_))) return rc_;
      } else if ((rc_ = tv_sweep_fused(h, f, h->v, P.lambda, clamp, (sw == 0 ? 1 : 0) | (sw == P.n_gd - 1 ? 2 : 0), s_))) return rc_;
    }
    if (P.n_gd == 0 && P.positivity && (rc_ = tv_clamp(h, f, s_))) return rc_;                     // Step 3 (:173)
    (void)it;
    return CTR_OK;
  };
  // The steady-state outer iteration - every steering scalar lives on the device, so its launch sequence is static -
  // is captured once into a CUDA graph and replayed: single problems are bound by launch latency (~150 kernels per
  // outer iteration of 1.9 ms at c3: 2.32 -> 1.92 ms), and 64 slices still gain 3 % (13.73 -> 13.33 ms: ~250 launches,
  // most of them short). The graph is keyed on the buffers and parameters baked into it; the event profiler
  // (ctr_profile_enable) turns it off.
  const bool graphs = !h->prof_on && !(h->g.flags & CTR_GEOM_NO_GRAPHS) && h->gstream;
  for (int it = 0; it < P.n_outer; ++it) {
    const bool x0_zero = it == 0 && !P.warm_start;
    const bool want_w = d_w && it == P.n_outer - 1;
    if (graphs && !x0_zero && !want_w) {
      GraphKey key;
      memset(&key, 0, sizeof(key));
      // (batched slices: the captured work reads and writes the handle's own buffers only)
      key.sino = direct ? d_sino : h->bsino; key.img = direct ? d_img : h->ximg; key.p = P; key.p.n_outer = 0; key.p.warm_start = 0; key.sel_k = h->sel_k;
      if (!h->graph_exec || memcmp(&key, &h->graph_key, sizeof(key)) != 0) {
        if (h->graph_exec) { cudaGraphExecDestroy(h->graph_exec); h->graph_exec = nullptr; }
        const long long l0 = h->launches, s0 = h->sweep_count;
        cudaGraph_t graph = nullptr;
        CTR_CUDA(h, cudaStreamBeginCapture(h->gstream, cudaStreamCaptureModeRelaxed));
        rc = outer(it, false, false, h->gstream);
        cudaError_t ce = cudaStreamEndCapture(h->gstream, &graph);
        h->graph_launches = h->launches - l0;
        h->launches = l0;          // nothing ran during the capture
        h->sweep_count = s0;
        if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
        if (ce != cudaSuccess) return cuda_fail(h, ce, "cudaStreamEndCapture");
        ce = cudaGraphInstantiate(&h->graph_exec, graph, 0);
        cudaGraphDestroy(graph);
        if (ce != cudaSuccess) { h->graph_exec = nullptr; return cuda_fail(h, ce, "cudaGraphInstantiate"); }
        h->graph_key = key;
      }
      CTR_CUDA(h, cudaGraphLaunch(h->graph_exec, st));
      h->launches += h->graph_launches;
      h->sweep_count += P.n_gd;
      continue;
    }
    if ((rc = outer(it, x0_zero, want_w, st))) return rc;
  }
  if (!direct && (rc = unpack(h, h->ximg, d_img, h->d.npix, 1, st))) return rc;
  if (d_w) {
    if (direct) CTR_CUDA(h, cudaMemcpyAsync(d_w, h->w, h->nimg * sizeof(float) * h->d.ndim, cudaMemcpyDeviceToDevice, st));
    else if ((rc = unpack(h, h->w, d_w, h->d.npix, h->d.ndim, st))) return rc;
  }
  return CTR_OK;
}

int ctr_reconstruct(ctr_handle* h, const float* d_sino, float* d_img, const ctr_params* p, void* stream) {
  return ctr_reconstruct_w(h, d_sino, d_img, nullptr, p, stream);
}

int ctr_profile_enable(ctr_handle* h, int on) {
  if (!h) return CTR_EINVAL;
  if (on && !h->prof_ev) {
    h->prof_ev = (cudaEvent_t*)calloc(2 * CTR_PROF_MAX, sizeof(cudaEvent_t));
    h->prof_kind = (unsigned char*)calloc(CTR_PROF_MAX, 1);
    if (!h->prof_ev || !h->prof_kind) return set_err(h, CTR_ENOMEM, "profiler allocation failed");
    for (int i = 0; i < 2 * CTR_PROF_MAX; ++i) CTR_CUDA(h, cudaEventCreate(&h->prof_ev[i]));
  }
  if (on) h->prof_n = 0;
  h->prof_on = on ? 1 : 0;
  return CTR_OK;
}

int ctr_profile_read(ctr_handle* h, double* ms_by_kind, long long* count_by_kind) {
  if (!h || !ms_by_kind || !count_by_kind) return CTR_EINVAL;
  CTR_CUDA(h, cudaStreamSynchronize(h->last_stream));
  for (int k = 0; k < CTR_PROF_KINDS; ++k) { ms_by_kind[k] = 0.0; count_by_kind[k] = 0; }
  for (int i = 0; i < h->prof_n; ++i) {
    float ms = 0.0f;
    CTR_CUDA(h, cudaEventElapsedTime(&ms, h->prof_ev[2 * i], h->prof_ev[2 * i + 1]));
    ms_by_kind[h->prof_kind[i]] += ms;
    count_by_kind[h->prof_kind[i]]++;
  }
  return CTR_OK;
}

int ctr_get_stats(ctr_handle* h, ctr_sweep_stat* buf, size_t n_records) {
  if (!h) return CTR_EINVAL;
  CTR_CUDA(h, cudaStreamSynchronize(h->last_stream));
  const int Bp = h->d.G * h->d.V, B = h->d.B;
  long long sweeps = h->sweep_count < CTR_STAT_SWEEPS ? h->sweep_count : CTR_STAT_SWEEPS;
  long long avail = sweeps * B;
  if (!buf || n_records == 0) return (int)avail;
  long long first = h->sweep_count - sweeps;
  size_t done = 0;
  for (long long sw = first; sw < h->sweep_count && done < n_records; ++sw) {
    size_t n = (size_t)B < n_records - done ? (size_t)B : n_records - done;
    CTR_CUDA(h, cudaMemcpy(buf + done, h->stats + (size_t)(sw % CTR_STAT_SWEEPS) * Bp, n * sizeof(ctr_sweep_stat),
                           cudaMemcpyDeviceToHost));
    done += n;
  }
  return (int)avail;
}

}  // extern "C"

