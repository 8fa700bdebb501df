// push_common.cuh -- device helpers shared by the order-1 and order-2 particle kernels.
#pragma once
#include "psc_internal.cuh"

// 1/sqrt(x) and 1/x for x >= 1 (1 + |u|^2, 1 + |t|^2): the bare MUFU approximations (2 ulp /
// 1 ulp), without the denormal-range scaling rsqrtf() and division wrap around them
__device__ __forceinline__ float rsqrt_ge1(float x) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float rcp_ge1(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// Boris rotation, PAPER.md:171-179 (Eq. 27-28): half electric kick, magnetic rotation with
// gamma taken after the first half kick ("We follow Boris"; A6), half electric kick.
// h = q dt / (2 m).  u is u = p/(m c).
__device__ __forceinline__ void boris_push(float &ux, float &uy, float &uz, float ex, float ey,
                                           float ez, float bx, float by, float bz, float h) {
  const float umx = fmaf(h, ex, ux), umy = fmaf(h, ey, uy), umz = fmaf(h, ez, uz);
  const float ig = h * rsqrt_ge1(fmaf(umx, umx, fmaf(umy, umy, fmaf(umz, umz, 1.0f))));
  const float tx = bx * ig, ty = by * ig, tz = bz * ig;
  const float sf = 2.0f * rcp_ge1(fmaf(tx, tx, fmaf(ty, ty, fmaf(tz, tz, 1.0f))));
  const float sx = tx * sf, sy = ty * sf, sz = tz * sf;
  const float upx = fmaf(umy, tz, fmaf(-umz, ty, umx));
  const float upy = fmaf(umz, tx, fmaf(-umx, tz, umy));
  const float upz = fmaf(umx, ty, fmaf(-umy, tx, umz));
  const float plx = fmaf(upy, sz, fmaf(-upz, sy, umx));
  const float ply = fmaf(upz, sx, fmaf(-upx, sz, umy));
  const float plz = fmaf(upx, sy, fmaf(-upy, sx, umz));
  ux = fmaf(h, ex, plx);
  uy = fmaf(h, ey, ply);
  uz = fmaf(h, ez, plz);
}

// streaming (read-once / write-once) particle column accesses: keep them out of L1
__device__ __forceinline__ float ld_stream(const float *p) { return __ldcs(p); }
__device__ __forceinline__ int ld_stream(const int *p) { return __ldcs(p); }
__device__ __forceinline__ void st_stream(float *p, float v) { __stcs(p, v); }
__device__ __forceinline__ void st_stream(int *p, int v) { __stcs(p, v); }

// asynchronous 4-byte global -> shared copy (LDGSTS); valid == false copies nothing and
// zero-fills the destination (src-size 0)
__device__ __forceinline__ void cp_async4(void *smem_dst, const void *gsrc, bool valid) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  const int sz = valid ? 4 : 0;
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(d), "l"(gsrc), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

__device__ __forceinline__ unsigned lanemask_lt_() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// Returns v, but opaque to the optimiser: what is computed from the result inside a loop stays
// inside the loop.  (Cheap per-cell recomputation of lane constants is deliberate: hoisted out of
// the particle loop they cost registers the loop needs, and end up spilled to local memory.)
__device__ __forceinline__ int keep_in_loop(int v) {
  asm volatile("" : "+r"(v));
  return v;
}
