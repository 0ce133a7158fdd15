// 3D circular cone-beam projector pair for sm_100a (config c5; the 3D extension of PAPER.md:85-89 by
// reading S22 -- Siddon's lengths are 3D by construction): ray-driven P (one thread per
// ray) and its exact transpose in gather form (one thread per voxel). As in 2D both evaluate ONE
// weight function (slab3_pieces) on ONE fp32 table, so the two matrices are bit-identical.
//
// Ray (view k, detector column a, row b) in grid-index coordinates, driving axis d in {x, y} (the
// in-plane axis it advances fastest along; the cone angle keeps |dz/dd| <= 1, checked at create):
//     o(d) = o0 + mo d      (other in-plane axis,  |mo| <= 1)       from table A[k][a]
//     z(d) = z0 + mz d      mz = vb q,  z0 = zs - mz ds,  vb = (b - boff_v) dv/dz   from table B[k][a]
// Within slab [s, s+1] of the driving axis the ray crosses at most one o grid line and at most one z
// grid plane, i.e. it visits at most three voxels; the slab's length L = sqrt(Lxy^2 + (mz dz)^2) is split
// at the two crossing parameters t_o, t_z in [0,1].
#include "ctr_common.cuh"
#include "ctr_internal.h"
#include "ctr_ell.cuh"

namespace ctr {

struct ConeGeomD {
  double dso, dsd, du, u_off, theta0, dtheta, xlo, ylo, zlo, dx, dy, dz;
  int nviews, nu, c0x, c0y, c0z;
};

// A = {o0, mo, +-Lxy, K = Lxy/|mo|},  B = {q = 1/(dD - dS), ds, zs, 1/|mo|}
__global__ void k_cone_build(ConeGeomD g, const float* __restrict__ angles, float4* __restrict__ A,
                             float4* __restrict__ B, float2* __restrict__ views) {
  int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= g.nviews * g.nu) return;
  int k = r / g.nu, a = r - k * g.nu;
  double th = angles ? (double)angles[k] : g.theta0 + g.dtheta * (double)k;
  double c = cos(th), s = sin(th);
  if (a == 0) views[k] = make_float2((float)c, (float)s);
  double Sx = -g.dso * c, Sy = -g.dso * s;
  double t = ((double)a - (g.nu - 1) / 2.0 + g.u_off) * g.du;
  double Dx = (g.dsd - g.dso) * c - t * s, Dy = (g.dsd - g.dso) * s + t * c;
  double sxp = (Sx - g.xlo) / g.dx - g.c0x, syp = (Sy - g.ylo) / g.dy - g.c0y;
  double dxp = (Dx - g.xlo) / g.dx - g.c0x, dyp = (Dy - g.ylo) / g.dy - g.c0y;
  double ddx = dxp - sxp, ddy = dyp - syp;
  bool xdrv = fabs(ddx) > fabs(ddy);
  double m, o0, L, dS, dD;
  if (!xdrv) {
    m = ddx / ddy; o0 = sxp - m * syp; L = sqrt(m * m * g.dx * g.dx + g.dy * g.dy); dS = syp; dD = dyp;
  } else {
    m = ddy / ddx; o0 = syp - m * sxp; L = sqrt(g.dx * g.dx + m * m * g.dy * g.dy); dS = sxp; dD = dxp;
  }
  float mf = (float)m;
  float K = (mf != 0.0f) ? (float)(L / fabs(m)) : 0.0f;
  float im = (mf != 0.0f) ? (float)(1.0 / fabs(m)) : 0.0f;
  A[r] = make_float4((float)o0, mf, xdrv ? -(float)L : (float)L, K);
  double zs = (0.0 - g.zlo) / g.dz - g.c0z;
  B[r] = make_float4((float)(1.0 / (dD - dS)), (float)dS, (float)zs, im);
}

// Everything both kernels need about one ray, derived with explicitly rounded operations so that the
// forward and the gather kernel get the same bits.
struct Ray3 {
  float o0, mo, z0, mz, L, inv_mo, inv_mz;
  bool xdrv;
};
__device__ __forceinline__ Ray3 cone_ray(const float4 A, const float4 B, int b, const Dims& d) {
  Ray3 r;
  r.o0 = A.x; r.mo = A.y; r.xdrv = A.z < 0.0f; r.inv_mo = B.w;
  const float vb = __fmul_rn(__fsub_rn((float)b, d.boff_v), d.dvz);
  r.mz = __fmul_rn(vb, B.x);
  r.z0 = fmaf(-r.mz, B.y, B.z);
  const float lz = __fmul_rn(r.mz, d.dz);
  r.L = __fsqrt_rn(fmaf(lz, lz, __fmul_rn(A.z, A.z)));
  r.inv_mz = r.mz != 0.0f ? __frcp_rn(fabsf(r.mz)) : 0.0f;
  return r;
}

// in-plane part of a slab (shared by all detector rows of a column)
struct SlabO {
  float ra, rb, t;  // biased entry / exit cell of the other axis, crossing parameter (1 if none)
};
__device__ __forceinline__ SlabO slab3_o(float oa, float ob, float inv_m) {
  SlabO s;
  s.ra = __fadd_rn(__fadd_rn(oa, -0.5f), CTR_MAGIC);
  s.rb = __fadd_rn(__fadd_rn(ob, -0.5f), CTR_MAGIC);
  const float Xc = __fadd_rn(fmaxf(s.ra, s.rb), -CTR_MAGIC);
  s.t = (s.ra == s.rb) ? 1.0f : fminf(__fmul_rn(fabsf(__fsub_rn(Xc, oa)), inv_m), 1.0f);
  return s;
}

// the (up to) three pieces of a slab: biased cells (po[i], pz[i]) and lengths w[i] in mm
struct Slab3 {
  float po[3], pz[3], w[3];
};
__device__ __forceinline__ Slab3 slab3_pieces(const SlabO so, const SlabO sz, float L) {
  Slab3 p;
  const float t1 = fminf(so.t, sz.t), t2 = fmaxf(so.t, sz.t);
  p.w[0] = __fmul_rn(L, t1);
  p.w[1] = __fmul_rn(L, __fsub_rn(t2, t1));
  p.w[2] = __fmul_rn(L, __fsub_rn(1.0f, t2));
  p.po[0] = so.ra; p.pz[0] = sz.ra;
  p.po[2] = so.rb; p.pz[2] = sz.rb;
  const bool o_first = so.t < sz.t;
  p.po[1] = o_first ? so.rb : so.ra;
  p.pz[1] = o_first ? sz.ra : sz.rb;
  return p;
}

// ------------------------------------------------------------------------------------------------
// a1 (3D)  P: one thread per ray; lanes of a warp are adjacent detector columns of one row.
// x-driving rays read the transposed copy volT[z][x][y]. MODEs as in the 2D kernel.
// ------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(128) k_cone_forward(Dims d, const float4* __restrict__ TA, const float4* __restrict__ TB,
                                                      const float* __restrict__ vol, const float* __restrict__ volT,
                                                      float* __restrict__ out, const float* __restrict__ bs, Scal sc,
                                                      double* part, unsigned* counter) {
  const int a = blockIdx.x * 128 + threadIdx.x;
  const int b = blockIdx.y, k = blockIdx.z;
  float acc = 0.0f;
  if (a < d.nu) {
    const int ka = k * d.nu + a;
    const Ray3 R = cone_ray(__ldg(&TA[ka]), __ldg(&TB[ka]), b, d);
    const int n_drv = R.xdrv ? d.nx : d.ny, n_oth = R.xdrv ? d.ny : d.nx;
    const int c_drv = R.xdrv ? d.c0x : d.c0y, c_oth = R.xdrv ? d.c0y : d.c0x;
    // slab range: the ray must be within one cell of the grid in both o and z
    float tlo = -1.0e6f, thi = 1.0e6f;
    {
      const float lo = (float)(-c_oth) - 1.0f, hi = (float)(n_oth - c_oth) + 1.0f;
      if (R.mo != 0.0f) {
        const float t1 = (lo - R.o0) / R.mo, t2 = (hi - R.o0) / R.mo;
        tlo = fmaxf(tlo, fminf(t1, t2)); thi = fminf(thi, fmaxf(t1, t2));
      } else if (R.o0 < lo || R.o0 > hi) thi = -2.0e6f;
      const float zl = (float)(-d.c0z) - 1.0f, zh = (float)(d.nz - d.c0z) + 1.0f;
      if (R.mz != 0.0f) {
        const float t1 = (zl - R.z0) / R.mz, t2 = (zh - R.z0) / R.mz;
        tlo = fmaxf(tlo, fminf(t1, t2)); thi = fminf(thi, fmaxf(t1, t2));
      } else if (R.z0 < zl || R.z0 > zh) thi = -2.0e6f;
    }
    int s0 = 0, s1 = 0;
    if (thi >= tlo) {
      s0 = max(0, (int)floorf(tlo) + c_drv - 2);
      s1 = min(n_drv, (int)ceilf(thi) + c_drv + 2);
    }
    const float* base = R.xdrv ? volT : vol;
    float y = (float)(s0 - c_drv);
    float oa = fmaf(R.mo, y, R.o0), za = fmaf(R.mz, y, R.z0);
    for (int s = s0; s < s1; ++s) {
      const float ob = fmaf(R.mo, y + 1.0f, R.o0), zb = fmaf(R.mz, y + 1.0f, R.z0);
      const Slab3 p = slab3_pieces(slab3_o(oa, ob, R.inv_mo), slab3_o(za, zb, R.inv_mz), R.L);
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        const int io = cell_of(p.po[q]) + c_oth, iz = cell_of(p.pz[q]) + d.c0z;
        if (p.w[q] != 0.0f && (unsigned)io < (unsigned)n_oth && (unsigned)iz < (unsigned)d.nz)
          acc = fmaf(p.w[q], __ldg(base + ((size_t)iz * n_drv + s) * n_oth + io), acc);
      }
      oa = ob; za = zb; y += 1.0f;
    }
    const size_t e = ((size_t)k * d.nv + b) * d.nu + a;
    if (MODE == 1) acc = __ldg(bs + e) - acc;
    out[e] = acc;
  }
  if (MODE == 2) {
    double v[1] = {(double)acc * (double)acc};
    const unsigned nblk = gridDim.x * gridDim.y * gridDim.z;
    const unsigned blk = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
    grid_reduce<1>(v, part, counter, nblk, blk, threadIdx.x, 128, [&](double(&sum)[1]) {
      const double gamma = sc.gamma[0];
      sc.a[0] = (sum[0] > 0.0 && gamma > 0.0) ? (float)(gamma / sum[0]) : 0.0f;  // S4
    });
  }
}

// ------------------------------------------------------------------------------------------------
// a2 (3D)  P^T (gather): one thread per voxel. Per view the candidate detector columns come from
// the in-plane window table of pixel (i,j) (exact first/last column with a non-zero in-plane
// weight, built at create); the candidate rows are a strict superset found by projecting the
// voxel's z-extent at the nearest / farthest in-plane distance. The in-plane part of the weight is
// evaluated once per column and reused for every row. No atomics, fixed accumulation order.
// ------------------------------------------------------------------------------------------------
// all rays with a non-zero weight in voxel (i, j, k), in a fixed order (views, columns, rows ascending):
// visit(ray index, p_ij)
template <class Visit>
__device__ __forceinline__ void cone_voxel_hits(const Dims& d, const float4* __restrict__ TA, const float4* __restrict__ TB,
                                                const float2* __restrict__ views, const unsigned short* __restrict__ win,
                                                int i, int j, int k, Visit visit) {
  const float fi = (float)(i - d.c0x), fj = (float)(j - d.c0y);
  const float bi = bias_of(i - d.c0x), bj = bias_of(j - d.c0y), bk = bias_of(k - d.c0z);
  const float px = fmaf((float)i + 0.5f, d.dx, d.xlo), py = fmaf((float)j + 0.5f, d.dy, d.ylo);
  const float z_lo = fmaf((float)k, d.dz, d.zlo), z_hi = z_lo + d.dz;  // voxel z-extent, mm
  const float rxy = 0.5f * sqrtf(d.dx * d.dx + d.dy * d.dy);
  const size_t pix = (size_t)j * d.nx + i;
  for (int kv = 0; kv < d.nviews; ++kv) {
    const unsigned w = __ldg(&win[(size_t)kv * d.nx * d.ny + pix]);
    const int a_lo = (int)(w >> 4), a_cnt = (int)(w & 15u);
    if (a_cnt == 0) continue;
    // detector rows: v = z dsd / den with den in [den_c - rxy, den_c + rxy]
    const float2 cs = __ldg(&views[kv]);
    const float den = fmaf(px, cs.x, fmaf(py, cs.y, d.dso));
    const float i1 = __frcp_rn(den - rxy) * d.dsd * d.inv_dv, i2 = __frcp_rn(den + rxy) * d.dsd * d.inv_dv;
    const float v1 = fminf(fminf(z_lo * i1, z_lo * i2), fminf(z_hi * i1, z_hi * i2));
    const float v2 = fmaxf(fmaxf(z_lo * i1, z_lo * i2), fmaxf(z_hi * i1, z_hi * i2));
    const int b_lo = max(0, (int)ceilf(v1 + d.boff_v - 0.05f));
    const int b_hi = min(d.nv - 1, (int)floorf(v2 + d.boff_v + 0.05f));
    for (int a = a_lo; a < a_lo + a_cnt; ++a) {
      const int ka = kv * d.nu + a;
      const float4 A = __ldg(&TA[ka]), B = __ldg(&TB[ka]);
      const bool xdrv = A.z < 0.0f;
      const float sc_ = xdrv ? fi : fj, tgt = xdrv ? bj : bi;
      const SlabO so = slab3_o(fmaf(A.y, sc_, A.x), fmaf(A.y, sc_ + 1.0f, A.x), B.w);
      if (so.ra != tgt && so.rb != tgt) continue;
      for (int b = b_lo; b <= b_hi; ++b) {
        const Ray3 R = cone_ray(A, B, b, d);
        const SlabO sz = slab3_o(fmaf(R.mz, sc_, R.z0), fmaf(R.mz, sc_ + 1.0f, R.z0), R.inv_mz);
        const Slab3 p = slab3_pieces(so, sz, R.L);
        float wt = 0.0f;
#pragma unroll
        for (int q = 0; q < 3; ++q) wt += (p.po[q] == tgt && p.pz[q] == bk) ? p.w[q] : 0.0f;
        if (wt != 0.0f) visit((kv * d.nv + b) * d.nu + a, wt);
      }
    }
  }
}

template <int MODE>
__global__ void __launch_bounds__(128) k_cone_back(Dims d, const float4* __restrict__ TA, const float4* __restrict__ TB,
                                                   const float2* __restrict__ views, const unsigned short* __restrict__ win,
                                                   const float* __restrict__ sino, float* __restrict__ out,
                                                   const float* __restrict__ s_img, float* __restrict__ u_img, Scal sc) {
  const int i = blockIdx.x * 32 + threadIdx.x;
  const int nby = (d.ny + 3) / 4;
  const int k = blockIdx.y / nby;
  const int j = (blockIdx.y - k * nby) * 4 + threadIdx.y;
  if (i >= d.nx || j >= d.ny) return;
  float acc = 0.0f;
  cone_voxel_hits(d, TA, TB, views, win, i, j, k, [&](int ray, float wt) { acc = fmaf(wt, __ldg(sino + ray), acc); });
  const size_t e = ((size_t)k * d.ny + j) * d.nx + i;
  out[e] = acc;
  if (MODE == 2) u_img[e] = fmaf(sc.a[0], __ldcg(s_img + e), __ldcg(u_img + e));
}

// ------------------------------------------------------------------------------------------------
// Row visitors for the stored matrices (ctr_ell.cuh): the same entries, in the same order, as the
// on-the-fly kernels above add them.
// ------------------------------------------------------------------------------------------------
struct ConeVoxelHits {  // rows of P^T: voxel (i, j, k), row = (k ny + j) nx + i; index = ray (kv nv + b) nu + a
  const float4 *TA, *TB;
  const float2* views;
  const unsigned short* win;
  template <class Visit>
  __device__ __forceinline__ void operator()(const Dims& d, size_t row, Visit visit) const {
    const int i = (int)(row % d.nx), j = (int)((row / d.nx) % d.ny), k = (int)(row / ((size_t)d.nx * d.ny));
    cone_voxel_hits(d, TA, TB, views, win, i, j, k, visit);
  }
};

struct ConeRayHits {  // rows of P: ray (k, b, a), row = (k nv + b) nu + a; index = voxel (iz ny + y) nx + x (blk: blk_index)
  const float4 *TA, *TB;
  int blk = 0;
  template <class Visit>
  __device__ __forceinline__ void operator()(const Dims& d, size_t row, Visit visit) const {
    const int a = (int)(row % d.nu), b = (int)((row / d.nu) % d.nv), k = (int)(row / ((size_t)d.nu * d.nv));
    const int ka = k * d.nu + a;
    const Ray3 R = cone_ray(__ldg(&TA[ka]), __ldg(&TB[ka]), b, d);
    const int n_drv = R.xdrv ? d.nx : d.ny, n_oth = R.xdrv ? d.ny : d.nx;
    const int c_drv = R.xdrv ? d.c0x : d.c0y, c_oth = R.xdrv ? d.c0y : d.c0x;
    float tlo = -1.0e6f, thi = 1.0e6f;
    {
      const float lo = (float)(-c_oth) - 1.0f, hi = (float)(n_oth - c_oth) + 1.0f;
      if (R.mo != 0.0f) {
        const float t1 = (lo - R.o0) / R.mo, t2 = (hi - R.o0) / R.mo;
        tlo = fmaxf(tlo, fminf(t1, t2)); thi = fminf(thi, fmaxf(t1, t2));
      } else if (R.o0 < lo || R.o0 > hi) thi = -2.0e6f;
      const float zl = (float)(-d.c0z) - 1.0f, zh = (float)(d.nz - d.c0z) + 1.0f;
      if (R.mz != 0.0f) {
        const float t1 = (zl - R.z0) / R.mz, t2 = (zh - R.z0) / R.mz;
        tlo = fmaxf(tlo, fminf(t1, t2)); thi = fminf(thi, fmaxf(t1, t2));
      } else if (R.z0 < zl || R.z0 > zh) thi = -2.0e6f;
    }
    int s0 = 0, s1 = 0;
    if (thi >= tlo) {
      s0 = max(0, (int)floorf(tlo) + c_drv - 2);
      s1 = min(n_drv, (int)ceilf(thi) + c_drv + 2);
    }
    float y = (float)(s0 - c_drv);
    float oa = fmaf(R.mo, y, R.o0), za = fmaf(R.mz, y, R.z0);
    for (int s = s0; s < s1; ++s) {
      const float ob = fmaf(R.mo, y + 1.0f, R.o0), zb = fmaf(R.mz, y + 1.0f, R.z0);
      const Slab3 p = slab3_pieces(slab3_o(oa, ob, R.inv_mo), slab3_o(za, zb, R.inv_mz), R.L);
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        const int io = cell_of(p.po[q]) + c_oth, iz = cell_of(p.pz[q]) + d.c0z;
        if (p.w[q] != 0.0f && (unsigned)io < (unsigned)n_oth && (unsigned)iz < (unsigned)d.nz)
        {
          const int px = R.xdrv ? s : io, py = R.xdrv ? io : s;
          visit(blk ? blk_index(px, py, iz, d.nx, d.ny) : (iz * d.ny + py) * d.nx + px, p.w[q]);
        }
      }
      oa = ob; za = zb; y += 1.0f;
    }
  }
};

// volT[z][x][y] = vol[z][y][x]
__global__ void __launch_bounds__(256) k_transpose3(int nx, int ny, const float* __restrict__ vol, float* __restrict__ volT) {
  __shared__ float tile[32][33];
  const size_t np = (size_t)nx * ny, zoff = (size_t)blockIdx.z * np;
  const int i0 = blockIdx.x * 32, j0 = blockIdx.y * 32;
  for (int r = threadIdx.y; r < 32; r += 8) {
    const int i = i0 + threadIdx.x, j = j0 + r;
    if (i < nx && j < ny) tile[r][threadIdx.x] = __ldcg(vol + zoff + (size_t)j * nx + i);
  }
  __syncthreads();
  for (int r = threadIdx.y; r < 32; r += 8) {
    const int j = j0 + threadIdx.x, i = i0 + r;
    if (i < nx && j < ny) volT[zoff + (size_t)i * ny + j] = tile[threadIdx.x][r];
  }
}

// in-plane window table for the gather (same encoding as the 2D table) + check |mz| <= 1
__global__ void __launch_bounds__(128) k_cone_window(Dims d, const float4* __restrict__ TA, const float4* __restrict__ TB,
                                                     const float2* __restrict__ views, unsigned short* __restrict__ win,
                                                     int* __restrict__ flags) {
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 4 + threadIdx.y, k = blockIdx.z;
  if (i >= d.nx || j >= d.ny) return;
  const float fi = (float)(i - d.c0x), fj = (float)(j - d.c0y);
  const float bi = bias_of(i - d.c0x), bj = bias_of(j - d.c0y);
  const float px = fmaf((float)i + 0.5f, d.dx, d.xlo), py = fmaf((float)j + 0.5f, d.dy, d.ylo);
  // conservative column window (in-plane, as fan_window with the in-plane half diagonal)
  const float2 cs = __ldg(&views[k]);
  const float rp = 0.5f * sqrtf(d.dx * d.dx + d.dy * d.dy), sdu = d.dsd * d.inv_du;
  const float den = fmaf(px, cs.x, fmaf(py, cs.y, d.dso)), aa = fmaf(py, cs.x, -px * cs.y);
  const float ell = sqrtf(aa * aa + den * den), inv = 1.0f / (den - rp);
  const float bc = fmaf(sdu * aa, 1.0f / den, d.boff_u), hb = rp * sdu * (ell + rp) * inv * inv;
  const int a_lo = max(0, (int)ceilf(bc - hb - 0.02f)), a_hi = min(d.nu - 1, (int)floorf(bc + hb + 0.02f));
  int first = -1, last = -2;
  for (int a = a_lo; a <= a_hi; ++a) {
    const float4 A = __ldg(&TA[k * d.nu + a]), B = __ldg(&TB[k * d.nu + a]);
    const bool xdrv = A.z < 0.0f;
    const float sc_ = xdrv ? fi : fj, tgt = xdrv ? bj : bi;
    const SlabO so = slab3_o(fmaf(A.y, sc_, A.x), fmaf(A.y, sc_ + 1.0f, A.x), B.w);
    if (so.ra == tgt || so.rb == tgt) {
      if (first < 0) first = a;
      last = a;
    }
    // largest |mz| of this column: detector rows 0 and nv-1
    const float m0 = fabsf((0.0f - d.boff_v) * d.dvz * B.x), m1 = fabsf(((float)(d.nv - 1) - d.boff_v) * d.dvz * B.x);
    if (fmaxf(m0, m1) > 1.0f) atomicExch(&flags[1], 1);
  }
  int cnt = last - first + 1;
  if (first < 0) { first = 0; cnt = 0; }
  if (cnt > 15 || first > 4095) { atomicExch(&flags[0], 1); cnt = 0; }
  win[(size_t)k * d.nx * d.ny + (size_t)j * d.nx + i] = (unsigned short)((first << 4) | cnt);
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
int cone_build_tables(ctr_handle* h) {
  const ctr_geometry& g = h->g;
  const Dims& d = h->d;
  ConeGeomD gd;
  gd.dso = g.dso; gd.dsd = g.dsd; gd.du = g.du; gd.u_off = g.u_off;
  gd.theta0 = g.theta0; gd.dtheta = g.dtheta;
  gd.dx = g.dx; gd.dy = g.dy; gd.dz = g.dz;
  gd.xlo = (double)g.cx - g.nx * (double)g.dx / 2.0;
  gd.ylo = (double)g.cy - g.ny * (double)g.dy / 2.0;
  gd.zlo = (double)g.cz - g.nz * (double)g.dz / 2.0;
  gd.nviews = g.nviews; gd.nu = g.nu; gd.c0x = d.c0x; gd.c0y = d.c0y; gd.c0z = d.c0z;
  float* d_angles = nullptr;
  if (g.angles) {
    CTR_CUDA(h, cudaMalloc(&d_angles, sizeof(float) * g.nviews));
    CTR_CUDA(h, cudaMemcpy(d_angles, g.angles, sizeof(float) * g.nviews, cudaMemcpyHostToDevice));
  }
  const int n = g.nviews * g.nu;
  k_cone_build<<<(n + 127) / 128, 128>>>(gd, d_angles, h->rays, h->rays2, h->views);
  CTR_LAUNCHED(h);
  int* d_flags = nullptr;
  CTR_CUDA(h, cudaMalloc(&d_flags, 2 * sizeof(int)));
  CTR_CUDA(h, cudaMemset(d_flags, 0, 2 * sizeof(int)));
  dim3 grid((d.nx + 31) / 32, (d.ny + 3) / 4, d.nviews), block(32, 4);
  k_cone_window<<<grid, block>>>(d, h->rays, h->rays2, h->views, h->win, d_flags);
  CTR_LAUNCHED(h);
  int flags[2] = {1, 1};
  CTR_CUDA(h, cudaMemcpy(flags, d_flags, sizeof(flags), cudaMemcpyDeviceToHost));
  cudaFree(d_flags);
  if (d_angles) cudaFree(d_angles);
  if (flags[0]) return set_err(h, CTR_EGEOM, "cone beam: a voxel sees more than 15 detector columns per view (or nu > 4095)");
  if (flags[1]) return set_err(h, CTR_EGEOM, "cone beam: a ray advances more than one voxel in z per in-plane voxel (|mz| > 1)");
  h->win_ok = 1;
  // stored matrices (best effort; ~40 GB each at c5)
  int rc = ell_build(h, ConeVoxelHits{h->rays, h->rays2, h->views, h->win}, (size_t)d.npix, h->ell_pt);
  // c5: ncu had the L1 data pipe 82 % busy with 9.5 wavefronts per warp gather in the row-major volume; with the blocked
  // copy the stored P takes 6.1 instead of 7.6 ms per application (DRAM-bound on its table, like P^T)
  h->ell_p_blk = (ELL_BLOCKED && blk_ok(d.nx, d.ny)) ? 1 : 0;
  if (rc == CTR_OK) rc = ell_build(h, ConeRayHits{h->rays, h->rays2, h->ell_p_blk}, (size_t)d.nray, h->ell_p);
  return rc;
}

int cone_forward(ctr_handle* h, const float* img, float* out, int mode, const float* bs, cudaStream_t st) {
  const Dims& d = h->d;
  ProfScope prof(h, CTR_PROF_FORWARD, st);
  if (h->ell_p.tab) {
    if (h->ell_p_blk) {
      k_to_blocked<<<(unsigned)((h->nimg + 255) / 256), 256, 0, st>>>(d.nx, d.ny, d.nz, img, h->imgT);
      CTR_LAUNCHED(h);
    }
    return ell_forward<1>(h, h->ell_p, h->ell_p_blk ? h->imgT : img, out, mode, bs, st);
  }
  {
    dim3 tg((d.nx + 31) / 32, (d.ny + 31) / 32, d.nz), tb(32, 8);
    k_transpose3<<<tg, tb, 0, st>>>(d.nx, d.ny, img, h->imgT);
    CTR_LAUNCHED(h);
  }
  dim3 grid((d.nu + 127) / 128, d.nv, d.nviews);
  if (mode == 0) k_cone_forward<0><<<grid, 128, 0, st>>>(d, h->rays, h->rays2, img, h->imgT, out, bs, h->sc, h->part, h->counters);
  else if (mode == 1) k_cone_forward<1><<<grid, 128, 0, st>>>(d, h->rays, h->rays2, img, h->imgT, out, bs, h->sc, h->part, h->counters);
  else k_cone_forward<2><<<grid, 128, 0, st>>>(d, h->rays, h->rays2, img, h->imgT, out, bs, h->sc, h->part, h->counters);
  CTR_LAUNCHED(h);
  return CTR_OK;
}

int cone_back(ctr_handle* h, const float* sino, float* out, int mode, const float* s, float* u, cudaStream_t st) {
  const Dims& d = h->d;
  ProfScope prof(h, CTR_PROF_BACK, st);
  dim3 grid((d.nx + 31) / 32, ((d.ny + 3) / 4) * d.nz), block(32, 4);
  if (h->ell_pt.tab) return ell_back(h, h->ell_pt, sino, out, mode, s, u, st);
  if (mode == 0) k_cone_back<0><<<grid, block, 0, st>>>(d, h->rays, h->rays2, h->views, h->win, sino, out, s, u, h->sc);
  else k_cone_back<2><<<grid, block, 0, st>>>(d, h->rays, h->rays2, h->views, h->win, sino, out, s, u, h->sc);
  CTR_LAUNCHED(h);
  return CTR_OK;
}

}  // namespace ctr
