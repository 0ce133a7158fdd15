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

}  // namespace ctr
