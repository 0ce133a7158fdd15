// 2D fan-beam projector pair for sm_100a: ray-driven P (one thread per ray and slice group)
// and its exact transpose P^T in gather form (one thread per pixel and slice group).
// Both evaluate the SAME slab_weights() on the SAME fp32 ray table, so every p_ij is identical
// bit for bit in the two kernels and <Px,y> = <x,P^T y> holds up to summation order.
//   P   : PAPER.md:87-89 (Eq. 1), :193 ("each thread responsible for one ray line")
//   P^T : PAPER.md:193 (why not scatter), :471 (adjoint condition A3'); north_star: exact transpose
#include "ctr_common.cuh"
#include "ctr_internal.h"
#include "ctr_fan_geom.cuh"
#include "ctr_ell.cuh"

namespace ctr {

// ------------------------------------------------------------------------------------------------
// Ray table, built once per handle in fp64 and rounded to fp32.
// Grid-index coordinates: X' = (x - xlo)/dx - c0x, so grid lines sit at integers -c0x .. nx-c0x.
//   y-driving (|dy'| >= |dx'|):  x'(y') = x0 + m y',  L = length per unit y' (mm), stored +L
//   x-driving:                    y'(x') = x0 + m x',  L = length per unit x' (mm), stored -L
//   K = L/|m| (0 when m = 0).
// ------------------------------------------------------------------------------------------------
struct FanGeomD {
  double dso, dsd, du, u_off, theta0, dtheta, xlo, ylo, dx, dy;
  int nviews, nu, c0x, c0y, det_type;
};

__global__ void k_fan_build(FanGeomD g, const float* __restrict__ angles, float4* __restrict__ rays,
                            float2* __restrict__ views, double2* __restrict__ viewsd) {
  int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= g.nviews * g.nu) return;
  int k = r / g.nu, b = r - k * g.nu;
  double th = angles ? (double)angles[k] : g.theta0 + g.dtheta * (double)k;
  double c = cos(th), s = sin(th);
  if (b == 0) {
    views[k] = make_float2((float)c, (float)s);
    viewsd[k] = make_double2(c, s);
  }
  double Sx = -g.dso * c, Sy = -g.dso * s;
  double t = ((double)b - (g.nu - 1) / 2.0 + g.u_off) * g.du;
  double Dx, Dy;
  if (g.det_type == 0) {
    Dx = (g.dsd - g.dso) * c - t * s;
    Dy = (g.dsd - g.dso) * s + t * c;
  } else {
    double beta = t / g.dsd;
    Dx = Sx + g.dsd * cos(th + beta);
    Dy = Sy + g.dsd * sin(th + beta);
  }
  double sxp = (Sx - g.xlo) / g.dx - g.c0x, syp = (Sy - g.ylo) / g.dy - g.c0y;
  double ddx = (Dx - Sx) / g.dx, ddy = (Dy - Sy) / g.dy;
  double m, x0, L;
  bool xdrv = fabs(ddx) > fabs(ddy);
  if (!xdrv) {
    m = ddx / ddy;
    x0 = sxp - m * syp;
    L = sqrt(m * m * g.dx * g.dx + g.dy * g.dy);
  } else {
    m = ddy / ddx;
    x0 = syp - m * sxp;
    L = sqrt(g.dx * g.dx + m * m * g.dy * g.dy);
  }
  float mf = (float)m;
  float K = (mf != 0.0f) ? (float)(L / fabs(m)) : 0.0f;
  rays[r] = make_float4((float)x0, mf, xdrv ? -(float)L : (float)L, K);
}

int fan_build_window(ctr_handle* h);

int fan_build_tables(ctr_handle* h) {
  const ctr_geometry& g = h->g;
  FanGeomD gd;
  gd.dso = g.dso; gd.dsd = g.dsd; gd.du = g.du; gd.u_off = g.u_off;
  gd.theta0 = g.theta0; gd.dtheta = g.dtheta;
  gd.dx = g.dx; gd.dy = g.dy;
  gd.xlo = (double)g.cx - g.nx * (double)g.dx / 2.0;
  gd.ylo = (double)g.cy - g.ny * (double)g.dy / 2.0;
  gd.nviews = g.nviews; gd.nu = g.nu; gd.c0x = h->d.c0x; gd.c0y = h->d.c0y; gd.det_type = g.det_type;
  float* d_angles = nullptr;
  if (g.angles) {
    CTR_CUDA(h, cudaMalloc(&d_angles, sizeof(float) * g.nviews));
    CTR_CUDA(h, cudaMemcpy(d_angles, g.angles, sizeof(float) * g.nviews, cudaMemcpyHostToDevice));
  }
  int n = g.nviews * g.nu;
  k_fan_build<<<(n + 127) / 128, 128>>>(gd, d_angles, h->rays, h->views, h->viewsd);
  CTR_LAUNCHED(h);
  CTR_CUDA(h, cudaDeviceSynchronize());
  if (d_angles) cudaFree(d_angles);
  return fan_build_window(h);
}

// Window table: win[view][pixel] = first_bin << 4 | count, the EXACT range of
// bins whose rays have a non-zero weight in the pixel, found once per handle by evaluating the
// weight function over the conservative window. overflow[0] is raised if a count exceeds 15.
__global__ void __launch_bounds__(128) k_fan_window(Dims d, const float4* __restrict__ rays,
                                                    const float2* __restrict__ views, unsigned short* __restrict__ win,
                                                    int* __restrict__ overflow) {
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 4 + threadIdx.y, k = blockIdx.z;
  if (i >= d.nx || j >= d.ny) return;
  const float fi = (float)(i - d.c0x), fj = (float)(j - d.c0y);
  const float bi = bias_of(i - d.c0x), bj = bias_of(j - d.c0y);
  const float px = fmaf((float)i + 0.5f, d.dx, d.xlo), py = fmaf((float)j + 0.5f, d.dy, d.ylo);
  int b_lo, b_hi, first = -1, last = -2;
  fan_window(d, __ldg(&views[k]), px, py, b_lo, b_hi);
  for (int b = b_lo; b <= b_hi; ++b) {
    if (fan_pixel_weight(__ldg(&rays[k * d.nu + b]), fi, fj, bi, bj) != 0.0f) {
      if (first < 0) first = b;
      last = b;
    }
  }
  int cnt = last - first + 1;
  if (first < 0) { first = 0; cnt = 0; }
  if (cnt > 15 || first > 4095) { atomicExch(overflow, 1); cnt = 0; }
  win[(size_t)k * d.npix + (size_t)j * d.nx + i] = (unsigned short)((first << 4) | cnt);
}

// win2[pixel][view] = win[view][pixel] (views contiguous: the batched gather takes LQ views per step)
__global__ void __launch_bounds__(256) k_win_transpose(const unsigned short* __restrict__ win,
                                                       unsigned short* __restrict__ win2, int npix, int nvp) {
  const int p = blockIdx.x * 256 + threadIdx.x, k = blockIdx.y;
  if (p < npix) win2[(size_t)p * nvp + k] = win[(size_t)k * npix + p];
}

// ------------------------------------------------------------------------------------------------
// Transposed copy imgT[g][i][j] = img[g][j][i] (32x32 tiles through shared memory). Rays whose driving
// axis is x walk columns of the image; reading them from the transposed copy makes their accesses as
// contiguous as those of y-driving rays (ncu, round 1: the forward projector was L1-wavefront bound).
// ------------------------------------------------------------------------------------------------
template <int V>
__global__ void __launch_bounds__(256) k_transpose(int nx, int ny, const float* __restrict__ img, float* __restrict__ imgT) {
  __shared__ float tile[32][33][V];
  const int g = blockIdx.z, i0 = blockIdx.x * 32, j0 = blockIdx.y * 32;
  const size_t np = (size_t)nx * ny;
  for (int r = threadIdx.y; r < 32; r += 8) {
    const int i = i0 + threadIdx.x, j = j0 + r;
    if (i < nx && j < ny) {
      float v[V];
      Pack<V>::ldcg(img, (size_t)g * np + (size_t)j * nx + i, v);
#pragma unroll
      for (int c = 0; c < V; ++c) tile[r][threadIdx.x][c] = v[c];
    }
  }
  __syncthreads();
  for (int r = threadIdx.y; r < 32; r += 8) {
    const int j = j0 + threadIdx.x, i = i0 + r;
    if (i < nx && j < ny) {
      float v[V];
#pragma unroll
      for (int c = 0; c < V; ++c) v[c] = tile[threadIdx.x][r][c];
      Pack<V>::st(imgT, (size_t)g * np + (size_t)i * ny + j, v);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// a1  P: one thread per ray and VG slice groups (V slices each). The thread walks the slabs of the
// ray's driving axis; per slab it touches at most two cells (|m| <= 1) and the geometry is shared by
// all V*VG slices. Lanes of a warp are adjacent bins of one view, so their cells are adjacent in
// memory (y-driving rays read img, x-driving rays read the transposed copy imgT).
// MODE 0: out = P x        MODE 1: out = bs - P x   (CGLS r0)
// MODE 2: out = P x and delta = ||out||^2 per slice -> a = gamma/delta (App. I step 1, :423)
// ------------------------------------------------------------------------------------------------
template <int V, int VG, int MODE>
__global__ void __launch_bounds__(128) k_fan_forward(Dims d, const float4* __restrict__ rays,
                                                     const float* __restrict__ img, const float* __restrict__ imgT,
                                                     float* __restrict__ out, const float* __restrict__ bs, Scal sc,
                                                     double* part, unsigned* counter) {
  const int r = blockIdx.x * 128 + threadIdx.x;
  const int g0 = blockIdx.y * VG;
  float acc[VG][V];
#pragma unroll
  for (int q = 0; q < VG; ++q)
#pragma unroll
    for (int c = 0; c < V; ++c) acc[q][c] = 0.0f;

  if (r < d.nray) {
    const float4 R = __ldg(&rays[r]);
    const float x0 = R.x, m = R.y, L = fabsf(R.z), K = R.w;
    const bool xdrv = R.z < 0.0f;
    const int n_drv = xdrv ? d.nx : d.ny, n_oth = xdrv ? d.ny : d.nx;
    const int c_drv = xdrv ? d.c0x : d.c0y, c_oth = xdrv ? d.c0y : d.c0x;
    // slabs in which the ray can be inside [-c_oth, n_oth - c_oth) (two cells of margin)
    int s0 = 0, s1 = n_drv;
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
    const float* base[VG];
#pragma unroll
    for (int q = 0; q < VG; ++q)
      base[q] = (xdrv ? imgT : img) + (size_t)min(g0 + q, d.G - 1) * d.npix * V;
    float y = (float)(s0 - c_drv);
    float oa = fmaf(m, y, x0);
    size_t row = (size_t)s0 * n_oth;
    for (int s = s0; s < s1; ++s) {
      const float ob = fmaf(m, y + 1.0f, x0);
      const SlabW w = slab_weights(oa, ob, L, K);
      const int ia = cell_of(w.ra) + c_oth, ib = cell_of(w.rb) + c_oth;
      if ((unsigned)ia < (unsigned)n_oth) {
#pragma unroll
        for (int q = 0; q < VG; ++q) {
          float f[V];
          Pack<V>::ld(base[q], row + ia, f);
#pragma unroll
          for (int c = 0; c < V; ++c) acc[q][c] = fmaf(w.wa, f[c], acc[q][c]);
        }
      }
      if (w.wb != 0.0f && (unsigned)ib < (unsigned)n_oth) {
#pragma unroll
        for (int q = 0; q < VG; ++q) {
          float f[V];
          Pack<V>::ld(base[q], row + ib, f);
#pragma unroll
          for (int c = 0; c < V; ++c) acc[q][c] = fmaf(w.wb, f[c], acc[q][c]);
        }
      }
      oa = ob;
      y += 1.0f;
      row += n_oth;
    }
#pragma unroll
    for (int q = 0; q < VG; ++q) {
      if (g0 + q < d.G) {
        const size_t e = (size_t)(g0 + q) * d.nray + r;
        if (MODE == 1) {
          float b[V];
          Pack<V>::ld(bs, e, b);
#pragma unroll
          for (int c = 0; c < V; ++c) acc[q][c] = b[c] - acc[q][c];
        }
        Pack<V>::st(out, e, acc[q]);
      }
    }
  }
  if (MODE == 2) {
    double v[VG * V];
#pragma unroll
    for (int q = 0; q < VG; ++q)
#pragma unroll
      for (int c = 0; c < V; ++c) v[q * V + c] = (double)acc[q][c] * (double)acc[q][c];
    grid_reduce<VG * V>(v, part + (size_t)blockIdx.y * gridDim.x * VG * V, counter + blockIdx.y, gridDim.x,
                        blockIdx.x, threadIdx.x, 128, [&](double(&sum)[VG * V]) {
#pragma unroll
                          for (int q = 0; q < VG; ++q)
#pragma unroll
                            for (int c = 0; c < V; ++c) {
                              if (g0 + q >= d.G) continue;
                              const int sl = (g0 + q) * V + c;
                              const double gamma = sc.gamma[sl];
                              sc.a[sl] = (sum[q * V + c] > 0.0 && gamma > 0.0) ? (float)(gamma / sum[q * V + c]) : 0.0f;  // S4
                            }
                        });
  }
}

// ------------------------------------------------------------------------------------------------
// a2  P^T (gather): one thread per pixel and VG slice groups. For every view the bins whose rays have
// a non-zero weight in the pixel come from the window table (TABLE = 1) or, if the table does not fit
// its 12+4-bit encoding, from fan_window(); slab_weights() gives exactly 0 for rays that miss.
// Accumulation order is fixed (views ascending, bins ascending); no atomics.
// MODE 0: out = P^T y
// MODE 2: out = g = P^T r and, fused, u += a s (App. I step 2) for the pixel it owns.
// (gamma, beta come from the re-orthogonalisation pass that follows, ctr_api.cu.)
// ------------------------------------------------------------------------------------------------
template <int V, int VG, int MODE, int TABLE>
__global__ void __launch_bounds__(128) k_fan_back(Dims d, const float4* __restrict__ rays,
                                                  const float2* __restrict__ views,
                                                  const unsigned short* __restrict__ win,
                                                  const float* __restrict__ sino, float* __restrict__ out,
                                                  const float* __restrict__ s_img, float* __restrict__ u_img, Scal sc) {
  const int i = blockIdx.x * 32 + threadIdx.x;
  const int j = blockIdx.y * 4 + threadIdx.y;
  const int g0 = blockIdx.z * VG;
  if (i >= d.nx || j >= d.ny) return;
  float acc[VG][V];
#pragma unroll
  for (int q = 0; q < VG; ++q)
#pragma unroll
    for (int c = 0; c < V; ++c) acc[q][c] = 0.0f;
  const float fi = (float)(i - d.c0x), fj = (float)(j - d.c0y);
  const float bi = bias_of(i - d.c0x), bj = bias_of(j - d.c0y);
  const float px = fmaf((float)i + 0.5f, d.dx, d.xlo), py = fmaf((float)j + 0.5f, d.dy, d.ylo);
  const size_t pix = (size_t)j * d.nx + i;
  const float* sg[VG];
#pragma unroll
  for (int q = 0; q < VG; ++q) sg[q] = sino + (size_t)min(g0 + q, d.G - 1) * d.nray * V;
  for (int k = 0; k < d.nviews; ++k) {
    int b_lo, b_hi;
    if (TABLE) {
      const unsigned w = __ldg(&win[(size_t)k * d.npix + pix]);
      b_lo = (int)(w >> 4);
      b_hi = b_lo + (int)(w & 15u) - 1;
    } else {
      fan_window(d, __ldg(&views[k]), px, py, b_lo, b_hi);
    }
    const int rbase = k * d.nu;
    for (int b = b_lo; b <= b_hi; ++b) {
      const float wt = fan_pixel_weight(__ldg(&rays[rbase + b]), fi, fj, bi, bj);
      if (wt != 0.0f) {
#pragma unroll
        for (int q = 0; q < VG; ++q) {
          float y[V];
          Pack<V>::ld(sg[q], (size_t)(rbase + b), y);
#pragma unroll
          for (int c = 0; c < V; ++c) acc[q][c] = fmaf(wt, y[c], acc[q][c]);
        }
      }
    }
  }
#pragma unroll
  for (int q = 0; q < VG; ++q) {
    if (g0 + q >= d.G) continue;
    const size_t e = (size_t)(g0 + q) * d.npix + pix;
    Pack<V>::st(out, e, acc[q]);
    if (MODE == 2) {
      float sv[V], uv[V];
      Pack<V>::ldcg(s_img, e, sv);
      Pack<V>::ldcg(u_img, e, uv);
#pragma unroll
      for (int c = 0; c < V; ++c) uv[c] = fmaf(sc.a[(g0 + q) * V + c], sv[c], uv[c]);
      Pack<V>::st(u_img, e, uv);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Row visitors for the stored matrices of a single slice (ctr_ell.cuh; the paper's lookup-table strategy,
// PAPER.md:193): the same entries, in the same order, as k_fan_forward<1,1,*> / k_fan_back<1,1,*> add them.
// ------------------------------------------------------------------------------------------------
#ifndef FAN_SPLIT
#define FAN_SPLIT 16 /* c3 forward per outer iteration: 1.05 / 0.96 / 0.91 / 1.05 ms for 4 / 8 / 16 / 32 */
#endif

// (FanRayHits, the row visitor of P, lives in ctr_fan_geom.cuh: the batched stored P of ctr_si.cu uses it too)

struct FanPixelHits {  // rows of P^T: pixel j nx + i; index = ray k nu + b
  const float4* rays;
  const float2* views;
  const unsigned short* win;
  int table;
  template <class Visit>
  __device__ __forceinline__ void operator()(const Dims& d, size_t row, Visit visit) const {
    const int i = (int)(row % d.nx), j = (int)(row / d.nx);
    const float fi = (float)(i - d.c0x), fj = (float)(j - d.c0y);
    const float bi = bias_of(i - d.c0x), bj = bias_of(j - d.c0y);
    const float px = fmaf((float)i + 0.5f, d.dx, d.xlo), py = fmaf((float)j + 0.5f, d.dy, d.ylo);
    for (int k = 0; k < d.nviews; ++k) {
      int b_lo, b_hi;
      if (table) {
        const unsigned w = __ldg(&win[(size_t)k * d.npix + row]);
        b_lo = (int)(w >> 4);
        b_hi = b_lo + (int)(w & 15u) - 1;
      } else {
        fan_window(d, __ldg(&views[k]), px, py, b_lo, b_hi);
      }
      for (int b = b_lo; b <= b_hi; ++b) {
        const float wt = fan_pixel_weight(__ldg(&rays[k * d.nu + b]), fi, fj, bi, bj);
        if (wt != 0.0f) visit(k * d.nu + b, wt);
      }
    }
  }
};

// ------------------------------------------------------------------------------------------------
// NEXT-1: the paper's own backprojector, Eq. (11) (App. III :467-493):
//   [P^T y](u*,v*) = (dx dy / dbeta) sum_theta y^theta(beta*) / l(u*,v*),  y^theta(beta*) by linear interpolation.
// One thread per pixel (as in the paper, :197) serving up to SC slices; the geometry of a (pixel, view) pair
// - fan angle, interpolation position, 1/(l dbeta) - is evaluated once in fp64 and shared by the slices;
// interpolation and accumulation in fp32. ARC: dbeta = du/dsd; FLAT: dbeta(beta*) = du cos^2(beta*)/dsd
// (reading S26). Works on the ABI arrays ([batch][nviews][nu] -> [batch][ny][nx]).
// ------------------------------------------------------------------------------------------------
template <int SC>
__global__ void __launch_bounds__(128) k_back_eq11(Dims d, double du, double u_off, const double2* __restrict__ viewsd,
                                                   const float* __restrict__ sino, float* __restrict__ img) {
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 4 + threadIdx.y;
  const int sl0 = blockIdx.z * SC;
  if (i >= d.nx || j >= d.ny) return;
  const double px = (double)d.xlo + ((double)i + 0.5) * (double)d.dx, py = (double)d.ylo + ((double)j + 0.5) * (double)d.dy;
  const double dso = (double)d.dso, dsd = (double)d.dsd, boff = (d.nu - 1) / 2.0 - u_off;
  float acc[SC];
#pragma unroll
  for (int c = 0; c < SC; ++c) acc[c] = 0.0f;
  const size_t sstride = (size_t)d.nviews * d.nu;
  for (int k = 0; k < d.nviews; ++k) {
    const double2 cs = viewsd[k];
    const double rx = px + dso * cs.x, ry = py + dso * cs.y;
    const double along = rx * cs.x + ry * cs.y, lateral = -rx * cs.y + ry * cs.x;
    const double l = sqrt(rx * rx + ry * ry);
    double bstar, dbeta;
    if (d.det_type == 1) {
      bstar = atan2(lateral, along) * dsd / du + boff;
      dbeta = du / dsd;
    } else {
      const double tb = lateral / along;  // tan(beta*)
      bstar = dsd * tb / du + boff;
      dbeta = du / (dsd * (1.0 + tb * tb));
    }
    if (!(along > 0.0) || !(bstar >= 0.0) || !(bstar <= (double)(d.nu - 1))) continue;
    int b0 = (int)floor(bstar);
    b0 = max(0, min(b0, d.nu - 2));
    const float fr = (float)(bstar - (double)b0), wgt = (float)(1.0 / (l * dbeta));
    const float* row = sino + (size_t)sl0 * sstride + (size_t)k * d.nu + b0;
#pragma unroll
    for (int c = 0; c < SC; ++c) {
      if (sl0 + c < d.B) {
        const float y0 = __ldg(row + c * sstride), y1 = d.nu > 1 ? __ldg(row + c * sstride + 1) : y0;
        acc[c] = fmaf(wgt, fmaf(fr, y1 - y0, y0), acc[c]);
      }
    }
  }
  const float scale = d.dx * d.dy;
#pragma unroll
  for (int c = 0; c < SC; ++c)
    if (sl0 + c < d.B) img[(size_t)(sl0 + c) * d.npix + (size_t)j * d.nx + i] = scale * acc[c];
}

int fan_back_eq11(ctr_handle* h, const float* sino, float* img, cudaStream_t st) {
  const Dims& d = h->d;
  ProfScope prof(h, CTR_PROF_BACK, st);
  dim3 block(32, 4);
  if (d.B == 1) {
    dim3 grid((d.nx + 31) / 32, (d.ny + 3) / 4, 1);
    k_back_eq11<1><<<grid, block, 0, st>>>(d, (double)h->g.du, (double)h->g.u_off, h->viewsd, sino, img);
  } else {
    dim3 grid((d.nx + 31) / 32, (d.ny + 3) / 4, (d.B + 7) / 8);
    k_back_eq11<8><<<grid, block, 0, st>>>(d, (double)h->g.du, (double)h->g.u_off, h->viewsd, sino, img);
  }
  CTR_LAUNCHED(h);
  return CTR_OK;
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
int fan_build_window(ctr_handle* h) {
  const Dims& d = h->d;
  h->win_ok = 0;
  if (d.nu > 4095) return CTR_OK;
  int* d_flag = nullptr;
  CTR_CUDA(h, cudaMalloc(&d_flag, sizeof(int)));
  CTR_CUDA(h, cudaMemset(d_flag, 0, sizeof(int)));
  dim3 grid((d.nx + 31) / 32, (d.ny + 3) / 4, d.nviews), block(32, 4);
  k_fan_window<<<grid, block>>>(d, h->rays, h->views, h->win, d_flag);
  CTR_LAUNCHED(h);
  int flag = 1;
  CTR_CUDA(h, cudaMemcpy(&flag, d_flag, sizeof(int), cudaMemcpyDeviceToHost));
  cudaFree(d_flag);
  h->win_ok = flag ? 0 : 1;
  if (h->win_ok && h->win2) {
    k_win_transpose<<<dim3((d.npix + 255) / 256, d.nviews), 256>>>(h->win, h->win2, d.npix, d.nvp);
    CTR_LAUNCHED(h);
    CTR_CUDA(h, cudaDeviceSynchronize());
  }
  if (d.V == 1) {
    // single slice: stored P and P^T (best effort). A ray's row has ~n entries and a slice has few rays:
    // each ray is dealt to FAN_SPLIT table rows (one thread each; c3: 198 us unsplit, 76 us on the fly, 57 us with 16 rows).
    // (the copy is one more launch per application: it pays from 512^2 on - c3 1.90 -> 1.885 ms, c2 0.546 -> 0.555 ms)
    h->ell_p_blk = (ELL_BLOCKED && blk_ok(d.nx, d.ny) && d.npix >= 512 * 512) ? 1 : 0;
    int rc = ell_build(h, SplitHits<FAN_SPLIT, FanRayHits>{FanRayHits{h->rays, h->ell_p_blk}}, (size_t)d.nray * FAN_SPLIT, h->ell_p);
    if (rc == CTR_OK) rc = ell_build(h, FanPixelHits{h->rays, h->views, h->win, h->win_ok}, (size_t)d.npix, h->ell_pt);
    return rc;
  }
  return CTR_OK;
}

template <int V, int VG>
static int fan_forward_v(ctr_handle* h, const float* img, float* out, int mode, const float* bs, cudaStream_t st) {
  const Dims& d = h->d;
  ProfScope prof(h, CTR_PROF_FORWARD, st);
  {
    dim3 tg((d.nx + 31) / 32, (d.ny + 31) / 32, d.G), tb(32, 8);
    k_transpose<V><<<tg, tb, 0, st>>>(d.nx, d.ny, img, h->imgT);
    CTR_LAUNCHED(h);
  }
  dim3 grid((d.nray + 127) / 128, (d.G + VG - 1) / VG);
  unsigned* cnt = h->counters + 0 * d.G;
  if (mode == 0) k_fan_forward<V, VG, 0><<<grid, 128, 0, st>>>(d, h->rays, img, h->imgT, out, bs, h->sc, h->part, cnt);
  else if (mode == 1) k_fan_forward<V, VG, 1><<<grid, 128, 0, st>>>(d, h->rays, img, h->imgT, out, bs, h->sc, h->part, cnt);
  else k_fan_forward<V, VG, 2><<<grid, 128, 0, st>>>(d, h->rays, img, h->imgT, out, bs, h->sc, h->part, cnt);
  CTR_LAUNCHED(h);
  return CTR_OK;
}

// batch == 1: the kernels above on the ABI arrays; batch > 1: slice-interleaved kernels of ctr_si.cu
int fan_forward(ctr_handle* h, const float* img, float* out, int mode, const float* bs, cudaStream_t st) {
  if (h->d.V == 1 && h->ell_p.tab) {
    const Dims& d = h->d;
    ProfScope prof(h, CTR_PROF_FORWARD, st);
    if (h->ell_p_blk) {
      k_to_blocked<<<(unsigned)((h->nimg + 255) / 256), 256, 0, st>>>(d.nx, d.ny, 1, img, h->imgT);
      CTR_LAUNCHED(h);
    }
    return ell_forward<FAN_SPLIT>(h, h->ell_p, h->ell_p_blk ? h->imgT : img, out, mode, bs, st);
  }
  if (h->d.V == 1) return fan_forward_v<1, 1>(h, img, out, mode, bs, st);
  return si_forward(h, img, out, mode, bs, st);
}

template <int V, int VG>
static int fan_back_v(ctr_handle* h, const float* sino, float* out, int mode, const float* s, float* u, cudaStream_t st) {
  const Dims& d = h->d;
  dim3 grid((d.nx + 31) / 32, (d.ny + 3) / 4, (d.G + VG - 1) / VG), block(32, 4);
  ProfScope prof(h, CTR_PROF_BACK, st);
#define CTR_BACK_LAUNCH(M, T) \
  k_fan_back<V, VG, M, T><<<grid, block, 0, st>>>(d, h->rays, h->views, h->win, sino, out, s, u, h->sc)
  if (h->win_ok) {
    if (mode == 0) CTR_BACK_LAUNCH(0, 1); else CTR_BACK_LAUNCH(2, 1);
  } else {
    if (mode == 0) CTR_BACK_LAUNCH(0, 0); else CTR_BACK_LAUNCH(2, 0);
  }
#undef CTR_BACK_LAUNCH
  CTR_LAUNCHED(h);
  return CTR_OK;
}

int fan_back(ctr_handle* h, const float* sino, float* out, int mode, const float* s, float* u, cudaStream_t st) {
  if (h->d.V == 1 && h->ell_pt.tab) {
    ProfScope prof(h, CTR_PROF_BACK, st);
    return ell_back(h, h->ell_pt, sino, out, mode, s, u, st);
  }
  if (h->d.V == 1) return fan_back_v<1, 1>(h, sino, out, mode, s, u, st);
  return si_back(h, sino, out, mode, s, u, st);
}

}  // namespace ctr

// =================================================================================================
// ctr_forward_noalloc (include/ctr.h): sino = P img for ONE 2D fan-beam slice without a handle and without any
// allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
// that forbid it). The kernels are the on-the-fly ones of ctr_forward (k_fan_build, k_transpose<1>, k_fan_forward<1,1,0>:
// identical bits); what a handle would own - the ray table and the transposed copy of the image - lives in a file-scope
// device array of fixed size, CTR_NOALLOC_SCRATCH_BYTES per GPU that loads the library, until the process exits.
// Every call uses that one array: calls that overlap on the GPU (two streams, two host threads) race. Nothing in
// it has to start at zero: each call overwrites rays[0, nray), views[0, nviews) and imgT[0, npix) before reading them.
// =================================================================================================
namespace {

struct NoallocScratch {
  float4 rays[CTR_NOALLOC_MAX_RAYS];      // ray table {x0, m, +-L, K}
  float imgT[CTR_NOALLOC_MAX_PIXELS];     // transposed copy of the image
  double2 viewsd[CTR_NOALLOC_MAX_VIEWS];  // (cos, sin) per view, written by k_fan_build
  float2 views[CTR_NOALLOC_MAX_VIEWS];
};
static_assert(sizeof(NoallocScratch) <= CTR_NOALLOC_SCRATCH_BYTES, "CTR_NOALLOC_SCRATCH_BYTES in include/ctr.h is too small");

static __device__ __align__(256) unsigned char g_noalloc_scratch[CTR_NOALLOC_SCRATCH_BYTES];

// In host code `g_noalloc_scratch` is only a host-side stand-in for the symbol: its device address is looked up once
// per device, with that device current, and cached here.
constexpr int NOALLOC_MAX_DEVICES = 64;
NoallocScratch* g_noalloc_ptr[NOALLOC_MAX_DEVICES];

int noalloc_scratch(int dev, NoallocScratch** out) {
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return CTR_ECUDA;
  if (!g_noalloc_ptr[dev]) {
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) { cudaGetLastError(); return CTR_ECUDA; }
    if (major != 10) return CTR_EARCH;
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) { cudaGetLastError(); return CTR_ECUDA; }
    g_noalloc_ptr[dev] = (NoallocScratch*)p;
  }
  *out = g_noalloc_ptr[dev];
  return CTR_OK;
}

}  // namespace

extern "C" int ctr_forward_noalloc(const ctr_geometry* g, const float* d_img, float* d_sino, void* stream) {
  using namespace ctr;
  if (!g || !d_img || !d_sino) return CTR_EINVAL;
  if ((((uintptr_t)d_img) | ((uintptr_t)d_sino)) & 15u) return CTR_EINVAL;
  if (g->ndim != 2 || g->nz != 1 || g->nv != 1 || g->batch != 1 || g->angles || g->flags) return CTR_EINVAL;
  if (g->nx < 1 || g->ny < 1 || g->nviews < 1 || g->nu < 1) return CTR_EINVAL;
  if (!(g->dx > 0) || !(g->dy > 0) || !(g->du > 0) || !(g->dso > 0) || !(g->dsd > g->dso)) return CTR_EINVAL;
  if (g->det_type != 0 && g->det_type != 1) return CTR_EINVAL;
  if ((long long)g->nx * g->ny > CTR_NOALLOC_MAX_PIXELS || (long long)g->nviews * g->nu > CTR_NOALLOC_MAX_RAYS ||
      g->nviews > CTR_NOALLOC_MAX_VIEWS)
    return CTR_ETOOBIG;
  {
    // same rule as ctr_create: source and detector outside the circle circumscribing the grid (plus one pixel)
    const double hx = fabs((double)g->cx) + 0.5 * g->nx * (double)g->dx + g->dx;
    const double hy = fabs((double)g->cy) + 0.5 * g->ny * (double)g->dy + g->dy;
    const double rad = sqrt(hx * hx + hy * hy);
    if (!(g->dso > rad) || !((double)g->dsd - g->dso > rad)) return CTR_EGEOM;
  }
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return CTR_ECUDA; }
  NoallocScratch* S = nullptr;
  int rc = noalloc_scratch(dev, &S);
  if (rc != CTR_OK) return rc;

  // problem description, as ctr_create fills it for a single 2D slice
  Dims d;
  memset(&d, 0, sizeof(d));
  d.ndim = 2;
  d.nx = g->nx; d.ny = g->ny; d.nz = 1;
  d.nviews = g->nviews; d.nu = g->nu; d.nv = 1;
  d.c0x = g->nx / 2; d.c0y = g->ny / 2; d.c0z = 0;
  d.npix = g->nx * g->ny;
  d.nray = g->nviews * g->nu;
  d.B = 1; d.V = 1; d.G = 1; d.GS = 1; d.LQ = 1;
  d.nvp = (g->nviews + 15) / 16 * 16;
  d.dx = g->dx; d.dy = g->dy; d.dz = 1.0f;
  d.xlo = (float)((double)g->cx - g->nx * (double)g->dx / 2.0);
  d.ylo = (float)((double)g->cy - g->ny * (double)g->dy / 2.0);
  d.zlo = -0.5f;
  d.dso = g->dso; d.dsd = g->dsd;
  d.inv_du = 1.0f / g->du; d.inv_dv = 1.0f; d.dvz = 1.0f;
  d.boff_u = (float)((g->nu - 1) / 2.0 - (double)g->u_off);
  d.boff_v = 0.0f;
  d.rvox = 0.5f * sqrtf(d.dx * d.dx + d.dy * d.dy);
  d.det_type = g->det_type;
  FanGeomD gd;
  gd.dso = g->dso; gd.dsd = g->dsd; gd.du = g->du; gd.u_off = g->u_off;
  gd.theta0 = g->theta0; gd.dtheta = g->dtheta;
  gd.dx = g->dx; gd.dy = g->dy;
  gd.xlo = (double)g->cx - g->nx * (double)g->dx / 2.0;
  gd.ylo = (double)g->cy - g->ny * (double)g->dy / 2.0;
  gd.nviews = g->nviews; gd.nu = g->nu; gd.c0x = d.c0x; gd.c0y = d.c0y; gd.det_type = g->det_type;

  cudaStream_t st = (cudaStream_t)stream;
  k_fan_build<<<(d.nray + 127) / 128, 128, 0, st>>>(gd, nullptr, S->rays, S->views, S->viewsd);
  k_transpose<1><<<dim3((d.nx + 31) / 32, (d.ny + 31) / 32, 1), dim3(32, 8), 0, st>>>(d.nx, d.ny, d_img, S->imgT);
  Scal none;
  memset(&none, 0, sizeof(none));
  k_fan_forward<1, 1, 0><<<dim3((d.nray + 127) / 128, 1), 128, 0, st>>>(d, S->rays, d_img, S->imgT, d_sino, nullptr, none,
                                                                        nullptr, nullptr);
  if (cudaPeekAtLastError() != cudaSuccess) { cudaGetLastError(); return CTR_ECUDA; }
  return CTR_OK;
}
