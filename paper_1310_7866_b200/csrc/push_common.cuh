// push_common.cuh -- device helpers shared by the order-1 and order-2 particle kernels.
#pragma once
#include "psc_internal.cuh"

// Boris rotation, PAPER.md:171-179 (Eq. 27-28): half electric kick, magnetic rotation with
// gamma taken after the first half kick ("We follow Boris"; A6), half electric kick.
// h = q dt / (2 m).  u is u = p/(m c).
__device__ __forceinline__ void boris_push(float &ux, float &uy, float &uz, float ex, float ey,
                                           float ez, float bx, float by, float bz, float h) {
  const float umx = fmaf(h, ex, ux), umy = fmaf(h, ey, uy), umz = fmaf(h, ez, uz);
  const float ig = h * rsqrtf(fmaf(umx, umx, fmaf(umy, umy, fmaf(umz, umz, 1.0f))));
  const float tx = bx * ig, ty = by * ig, tz = bz * ig;
  const float sf = __fdividef(2.0f, fmaf(tx, tx, fmaf(ty, ty, fmaf(tz, tz, 1.0f))));
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

__device__ __forceinline__ unsigned lanemask_lt_() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// Per-warp bookkeeping of the direction codes of one cell's particles (9 / 27
// destination classes): the stayers are counted with a ballot, the few leavers with
// shared-memory integer atomics on the warp's private row.  cell_done() writes the cell's ND
// counts (what the index sort of sort.cu consumes) and clears the row.
template <bool D3>
struct DirCount {
  static constexpr int ND = D3 ? 27 : 9, STAY = D3 ? 13 : 4;
  int *row;   // shared, [32], zero on entry
  int nstay;
  __device__ __forceinline__ void init(int *r, int lane) {
    row = r;
    row[lane] = 0;
    nstay = 0;
    __syncwarp();
  }
  __device__ __forceinline__ void add(bool act, int dc) {
    const bool stay = dc == STAY;
    nstay += __popc(__ballot_sync(0xffffffffu, act && stay));
    if (act && !stay) atomicAdd(&row[dc], 1);
  }
  __device__ __forceinline__ void cell_done(int *__restrict__ dircnt, int key, int lane) {
    __syncwarp();
    if (lane < ND) {
      dircnt[key * ND + lane] = row[lane] + (lane == STAY ? nstay : 0);
      row[lane] = 0;
    }
    nstay = 0;
    __syncwarp();
  }
};
