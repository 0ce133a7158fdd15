// Pixel-side geometry of the 2D fan beam shared by the gather backprojectors (ctr_fan.cu, ctr_si.cu).
#pragma once
#include "ctr_common.cuh"
#include "ctr_internal.h"

namespace ctr {

// ------------------------------------------------------------------------------------------------
// Candidate bins of a pixel in one view: rays that can cross the pixel project into a short window
// around the projection of its centre. The half width is a strict bound (half diagonal of the pixel
// times the largest magnification over the pixel) plus a guard, so approximate reciprocals are fine.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void fan_window(const Dims& d, float2 cs, float px, float py, int& b_lo, int& b_hi) {
  const float rp = d.rvox, sdu = d.dsd * d.inv_du;
  const float den = fmaf(px, cs.x, fmaf(py, cs.y, d.dso));  // distance along the central ray
  const float aa = fmaf(py, cs.x, -px * cs.y);              // lateral offset
  const float ell = aa * aa + den * den;
  float bc, hb;
  if (d.det_type == 0) {
    const float inv = __frcp_rn(den - rp);
    bc = fmaf(sdu * aa, __frcp_rn(den), d.boff_u);
    hb = rp * sdu * (ell * rsqrtf(ell) + rp) * inv * inv;
  } else {
    bc = fmaf(atan2f(aa, den), sdu, d.boff_u);
    hb = rp * sdu * __frcp_rn(ell * rsqrtf(ell) - rp);
  }
  b_lo = max(0, (int)ceilf(bc - hb - 0.02f));
  b_hi = min(d.nu - 1, (int)floorf(bc + hb + 0.02f));
}

// weight of ray R in pixel (cell coordinates fi,fj / biased bi,bj): the gather side of slab_weights()
__device__ __forceinline__ float fan_pixel_weight(const float4 R, float fi, float fj, float bi, float bj) {
  const bool xdrv = R.z < 0.0f;
  const float sc_ = xdrv ? fi : fj, tgt = xdrv ? bj : bi;
  const float oa = fmaf(R.y, sc_, R.x);
  const float ob = fmaf(R.y, sc_ + 1.0f, R.x);
  const SlabW w = slab_weights(oa, ob, fabsf(R.z), R.w);
  return (w.ra == tgt ? w.wa : 0.0f) + (w.rb == tgt ? w.wb : 0.0f);
}

// Row visitor of P: every non-zero (pixel index j nx + i, p_ij) of ray `row`, slab by slab, exactly the entries and
// the order k_fan_forward adds them in (stored matrices: ctr_ell.cuh for single slices, k_si_forward_tab for batches).
// Blocked copy of an image / volume for the gathers of the stored P of single problems (ctr_ell.cuh): 4 (y) x 8 (x)
// tiles of 32 floats = one 128-byte line each, [z][ny/4][nx/8][4][8]. The threads of a warp gather from neighbouring
// rays (3D) or from consecutive slabs of one ray (2D): in the row-major image that is one line per thread whenever
// the neighbours differ in y, in the blocked copy a handful of lines for either orientation.
__host__ __device__ __forceinline__ bool blk_ok(int nx, int ny) { return nx % 8 == 0 && ny % 4 == 0; }
__device__ __forceinline__ int blk_index(int x, int y, int z, int nx, int ny) {
  return (((z * (ny >> 2) + (y >> 2)) * (nx >> 3) + (x >> 3)) << 5) + ((y & 3) << 3) + (x & 7);
}

struct FanRayHits {  // rows of P: ray r = k nu + b; index = pixel j nx + i (blk != 0: blk_index of it)
  const float4* rays;
  int blk = 0;
  template <class Visit>
  __device__ __forceinline__ void operator()(const Dims& d, size_t row, Visit visit) const {
    const float4 R = __ldg(&rays[row]);
    const float x0 = R.x, m = R.y, L = fabsf(R.z), K = R.w;
    const bool xdrv = R.z < 0.0f;
    const int n_drv = xdrv ? d.nx : d.ny, n_oth = xdrv ? d.ny : d.nx;
    const int c_drv = xdrv ? d.c0x : d.c0y, c_oth = xdrv ? d.c0y : d.c0x;
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
    float y = (float)(s0 - c_drv);
    float oa = fmaf(m, y, x0);
    for (int s = s0; s < s1; ++s) {
      const float ob = fmaf(m, y + 1.0f, x0);
      const SlabW w = slab_weights(oa, ob, L, K);
      const int ia = cell_of(w.ra) + c_oth, ib = cell_of(w.rb) + c_oth;
      if (w.wa != 0.0f && (unsigned)ia < (unsigned)n_oth) {
        const int px = xdrv ? s : ia, py = xdrv ? ia : s;
        visit(blk ? blk_index(px, py, 0, d.nx, d.ny) : py * d.nx + px, w.wa);
      }
      if (w.wb != 0.0f && (unsigned)ib < (unsigned)n_oth) {
        const int px = xdrv ? s : ib, py = xdrv ? ib : s;
        visit(blk ? blk_index(px, py, 0, d.nx, d.ny) : py * d.nx + px, w.wb);
      }
      oa = ob;
      y += 1.0f;
    }
  }
};

}  // namespace ctr
