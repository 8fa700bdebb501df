// push_common.cuh -- device helpers shared by the order-1 and order-2 particle kernels.
#pragma once
#include "psc_internal.cuh"

// Boris rotation, PAPER.md:171-179 (Eq. 27-28): half electric kick, magnetic rotation with
// gamma taken after the first half kick ("We follow Boris"; A6), half electric kick.
// h = q dt / (2 m).  u is u = p/(m c).
__device__ __forceinline__ void boris_push(float &ux, float &uy, float &uz, float ex, float ey,
                                           float ez, float bx, float by, float bz, float h) {
  const float umx = fmaf(h, ex, ux), umy = fmaf(h, ey, uy), umz = fmaf(h, ez, uz);
  const float ig = h * rsqrtf(1.0f + umx * umx + umy * umy + umz * umz);
  const float tx = bx * ig, ty = by * ig, tz = bz * ig;
  const float sf = 2.0f / (1.0f + tx * tx + ty * ty + tz * tz);
  const float sx = tx * sf, sy = ty * sf, sz = tz * sf;
  const float upx = umx + (umy * tz - umz * ty);
  const float upy = umy + (umz * tx - umx * tz);
  const float upz = umz + (umx * ty - umy * tx);
  const float plx = umx + (upy * sz - upz * sy);
  const float ply = umy + (upz * sx - upx * sz);
  const float plz = umz + (upx * sy - upy * sx);
  ux = fmaf(h, ex, plx);
  uy = fmaf(h, ey, ply);
  uz = fmaf(h, ez, plz);
}

// streaming (read-once / write-once) particle column accesses: keep them out of L1
__device__ __forceinline__ float ld_stream(const float *p) { return __ldcs(p); }
__device__ __forceinline__ int ld_stream(const int *p) { return __ldcs(p); }
__device__ __forceinline__ void st_stream(float *p, float v) { __stcs(p, v); }
