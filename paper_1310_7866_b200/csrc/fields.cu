// fields.cu -- Yee-grid FDTD half/full steps and the single-GPU ghost operations.
//
// PAPER.md:98-160 (Eq. 12-18): B -= h curl+ E (forward differences), E += h (curl- B - J)
// (backward differences), leap-frog in time as in Fig. 8.
// fill_ghosts / add_and_fill_ghosts; on one GPU with periodic
// boundaries a ghost point is the periodic image of an interior point.
//
// Every kernel here is a pure streaming stencil over the [3][ez][ey][ex] arrays (x fastest):
// one thread per grid point handles the three components, loads are coalesced along the
// fastest non-trivial direction, and a thread writes only its own point, so the update kernels
// can write interior AND ghost points in one launch (a ghost point repeats the arithmetic of its
// image on identical values, hence stays bit-identical to it) -- no separate ghost-fill pass.
#include "psc_internal.cuh"

namespace {

struct Pt {
  int c[3];
  int idx;
};

__device__ __forceinline__ Pt decode(const GridDesc &gd, int idx) {
  Pt p;
  p.idx = idx;
  p.c[0] = idx % gd.ext[0];
  int r = idx / gd.ext[0];
  p.c[1] = r % gd.ext[1];
  p.c[2] = r / gd.ext[1];
  return p;
}

// offset to the +1 neighbour along d, wrapped periodically inside the extended array
__device__ __forceinline__ int up(const GridDesc &gd, const Pt &p, int d) {
  return (p.c[d] + 1 < gd.ext[d]) ? gd.nbo[d] : -(gd.n[d] - 1) * gd.nbo[d];
}
__device__ __forceinline__ int down(const GridDesc &gd, const Pt &p, int d) {
  return (p.c[d] > 0) ? -gd.nbo[d] : (gd.n[d] - 1) * gd.nbo[d];
}

// B -= h * curl+ E    (Eq. 12, 18)
__global__ void __launch_bounds__(256) k_push_b(GridDesc gd, const float *__restrict__ E,
                                                float *__restrict__ B, float hx, float hy,
                                                float hz) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= gd.comp) return;
  const Pt p = decode(gd, idx);
  const int ux = up(gd, p, 0), uy = up(gd, p, 1), uz = up(gd, p, 2);
  const float *Ex = E, *Ey = E + gd.comp, *Ez = E + 2 * gd.comp;
  const float ex = Ex[idx], ey = Ey[idx], ez = Ez[idx];
  float bx = B[idx], by = B[idx + gd.comp], bz = B[idx + 2 * gd.comp];
  bx -= hy * (Ez[idx + uy] - ez) - hz * (Ey[idx + uz] - ey);
  by -= hz * (Ex[idx + uz] - ex) - hx * (Ez[idx + ux] - ez);
  bz -= hx * (Ey[idx + ux] - ey) - hy * (Ex[idx + uy] - ex);
  B[idx] = bx;
  B[idx + gd.comp] = by;
  B[idx + 2 * gd.comp] = bz;
}

// E += h * (curl- B - J)    (Eq. 13, 17; c = eps0 = 1)
__global__ void __launch_bounds__(256) k_push_e(GridDesc gd, float *__restrict__ E,
                                                const float *__restrict__ B,
                                                const float *__restrict__ J, float hx, float hy,
                                                float hz, float h) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= gd.comp) return;
  const Pt p = decode(gd, idx);
  const int dx = down(gd, p, 0), dy = down(gd, p, 1), dz = down(gd, p, 2);
  const float *Bx = B, *By = B + gd.comp, *Bz = B + 2 * gd.comp;
  const float bx = Bx[idx], by = By[idx], bz = Bz[idx];
  float ex = E[idx], ey = E[idx + gd.comp], ez = E[idx + 2 * gd.comp];
  ex += hy * (bz - Bz[idx + dy]) - hz * (by - By[idx + dz]) - h * J[idx];
  ey += hz * (bx - Bx[idx + dz]) - hx * (bz - Bz[idx + dx]) - h * J[idx + gd.comp];
  ez += hx * (by - By[idx + dx]) - hy * (bx - Bx[idx + dy]) - h * J[idx + 2 * gd.comp];
  E[idx] = ex;
  E[idx + gd.comp] = ey;
  E[idx + 2 * gd.comp] = ez;
}

// ghosts := periodic images of the interior
__global__ void __launch_bounds__(256) k_fill_ghosts(GridDesc gd, float *__restrict__ F) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= gd.comp) return;
  const Pt p = decode(gd, idx);
  int src = idx;
  bool ghost = false;
#pragma unroll
  for (int d = 0; d < 3; d++) {
    if (p.c[d] < gd.g[d]) {
      src += gd.n[d] * gd.st[d];
      ghost = true;
    } else if (p.c[d] >= gd.g[d] + gd.n[d]) {
      src -= gd.n[d] * gd.st[d];
      ghost = true;
    }
  }
  if (!ghost) return;
#pragma unroll
  for (int c = 0; c < 3; c++) F[idx + c * gd.comp] = F[src + c * gd.comp];
}

// interior += every ghost image of it (add_ghosts).  Reads ghosts and the
// thread's own interior point, writes only that point: race free in one launch.
__global__ void __launch_bounds__(256) k_fold(GridDesc gd, float *__restrict__ F) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= gd.comp) return;
  const Pt p = decode(gd, idx);
  int sh[3];
#pragma unroll
  for (int d = 0; d < 3; d++) {
    const int ii = p.c[d] - gd.g[d];
    if (ii < 0 || ii >= gd.n[d]) return;  // ghost point: nothing to do
    sh[d] = 0;
    if (ii < gd.g[d])
      sh[d] = gd.n[d] * gd.st[d];  // image in the high ghost layers
    else if (ii >= gd.n[d] - gd.g[d])
      sh[d] = -gd.n[d] * gd.st[d];  // image in the low ghost layers
  }
  if ((sh[0] | sh[1] | sh[2]) == 0) return;
  float a0 = 0.f, a1 = 0.f, a2 = 0.f;
#pragma unroll
  for (int m = 1; m < 8; m++) {
    bool ok = true;
    int off = 0;
#pragma unroll
    for (int d = 0; d < 3; d++)
      if (m & (1 << d)) {
        if (sh[d] == 0) ok = false;
        off += sh[d];
      }
    if (ok) {
      a0 += F[idx + off];
      a1 += F[idx + off + gd.comp];
      a2 += F[idx + off + 2 * gd.comp];
    }
  }
  F[idx] += a0;
  F[idx + gd.comp] += a1;
  F[idx + 2 * gd.comp] += a2;
}

}  // namespace

int psc_fields_push_b(psc_ctx *c, float frac, cudaStream_t s) {
  const GridDesc &gd = c->gd;
  const float h = frac * gd.dt;
  const int blocks = (int)cdiv64(gd.comp, 256);
  k_push_b<<<blocks, 256, 0, s>>>(gd, c->E, c->B, gd.n[0] > 1 ? h * gd.inv_dx[0] : 0.f,
                                  gd.n[1] > 1 ? h * gd.inv_dx[1] : 0.f,
                                  gd.n[2] > 1 ? h * gd.inv_dx[2] : 0.f);
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}

int psc_fields_push_e(psc_ctx *c, float frac, cudaStream_t s) {
  const GridDesc &gd = c->gd;
  const float h = frac * gd.dt;
  const int blocks = (int)cdiv64(gd.comp, 256);
  k_push_e<<<blocks, 256, 0, s>>>(gd, c->E, c->B, c->J, gd.n[0] > 1 ? h * gd.inv_dx[0] : 0.f,
                                  gd.n[1] > 1 ? h * gd.inv_dx[1] : 0.f,
                                  gd.n[2] > 1 ? h * gd.inv_dx[2] : 0.f, h);
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}

int psc_fields_fill_ghosts(psc_ctx *c, float *F, cudaStream_t s) {
  const int blocks = (int)cdiv64(c->gd.comp, 256);
  k_fill_ghosts<<<blocks, 256, 0, s>>>(c->gd, F);
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}

int psc_fields_fold(psc_ctx *c, float *F, cudaStream_t s) {
  const int blocks = (int)cdiv64(c->gd.comp, 256);
  k_fold<<<blocks, 256, 0, s>>>(c->gd, F);
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}
