// marder.cu -- node charge density and Marder's Gauss-law correction.
//
// "single precision simulations that run for a very large number of steps accumulate round-off
// errors that lead to growing deviations from the discrete Gauss's Law.  PSC implements the
// iterative method by Marder to dissipate violations of Gauss's Law."  The paper only cites the
// method; the reading (A28) is one diffusion pass per iteration,
//   f = div- E - rho  on the nodes (Eq. 16, 24),      E <- E + D grad+ f,
// with (grad+ f)_x,i+1/2 = (f[i+1] - f[i]) / dx, so that the residual obeys f <- f + D lap f with
// the 7-point Laplacian div- grad+: every Fourier mode shrinks by 1 - D sum_d K_d^2 per pass,
// monotonically as long as D sum_d 4/dx_d^2 <= 1 (checked by psc_marder).
//
// rho sits on the nodes ("charge densities on corners") and is the particles' charge
// weighted with the same b1 / b2 the gather uses (A1).  It is deposited from the cell
// store: a warp per cell sums the stencil weights of the cell's residents in registers (the
// stencil nodes are the same for all of them), reduces across lanes and issues one global atomic
// per node; the records waiting in the cell's exchange row belong to neighbouring cells and are
// added record by record.
#include "store.cuh"

#include <mutex>

namespace {

constexpr int MT = 256;

__device__ __forceinline__ void key_to_cell3(const GridDesc &gd, int k, int c[3]) {
  const int b = k / gd.cpb, l = k - b * gd.cpb;
  const int b0 = b % gd.nb[0], br = b / gd.nb[0];
  const int b1 = br % gd.nb[1], b2 = br / gd.nb[1];
  const int l0 = l % gd.bs[0], lr = l / gd.bs[0];
  const int l1 = lr % gd.bs[1], l2 = lr / gd.bs[1];
  c[0] = b0 * gd.bs[0] + l0;
  c[1] = b1 * gd.bs[1] + l1;
  c[2] = b2 * gd.bs[2] + l2;
}

// weights of offset a in [0,1) on the NW nodes of one direction: order 1: nodes l, l+1 (b1);
// order 2: nodes l-1 .. l+2 (b2, Eq. 31; three of the four are non-zero)
template <int ORDER>
__device__ __forceinline__ void node_weights(float a, float (&w)[ORDER == 1 ? 2 : 4]) {
  if (ORDER == 1) {
    w[0] = 1.f - a;
    w[1] = a;
  } else {
    const bool up = a >= 0.5f;
    const float h = up ? a - 1.0f : a;
    const float wm = 0.5f * (0.5f - h) * (0.5f - h), w0 = 0.75f - h * h, wp = 0.5f * (0.5f + h) * (0.5f + h);
    w[0] = up ? 0.f : wm;
    w[1] = up ? wm : w0;
    w[2] = up ? w0 : wp;
    w[3] = up ? wp : 0.f;
  }
}

template <bool D3, int ORDER>
__global__ void __launch_bounds__(MT)
k_rho(GridDesc gd, Cols in, const int *__restrict__ base, const int *__restrict__ cnt, Exchange xin,
      float *__restrict__ rho) {
  constexpr int NW = ORDER == 1 ? 2 : 4, J0 = ORDER == 1 ? 0 : -1;
  constexpr int NN = D3 ? NW * NW * NW : NW * NW;
  constexpr int XW = D3 ? PSC_XW3 : PSC_XW2, ND = D3 ? 27 : 9;
  const int lane = threadIdx.x & 31;
  const int warps = gridDim.x * (MT / 32);
  for (int k = blockIdx.x * (MT / 32) + (threadIdx.x >> 5); k < gd.nkeys; k += warps) {
    int c[3];
    key_to_cell3(gd, k, c);
    const int n = cnt[k];
    const size_t b = (size_t)base[k];
    float acc[NN];
#pragma unroll
    for (int i = 0; i < NN; i++) acc[i] = 0.f;
    for (int v = lane; v < n; v += 32) {
      const float q = in.qw[b + v] * gd.inv_dV;
      float wx[NW], wy[NW], wz[NW];
      if (D3) node_weights<ORDER>(in.x[b + v], wx);
      node_weights<ORDER>(in.y[b + v], wy);
      node_weights<ORDER>(in.z[b + v], wz);
#pragma unroll
      for (int jz = 0; jz < NW; jz++)
#pragma unroll
        for (int jy = 0; jy < NW; jy++) {
          const float t = q * wz[jz] * wy[jy];
          if (D3) {
#pragma unroll
            for (int jx = 0; jx < NW; jx++) acc[(jz * NW + jy) * NW + jx] += t * wx[jx];
          } else {
            acc[jz * NW + jy] += t;
          }
        }
    }
    if (n > 0) {
#pragma unroll
      for (int i = 0; i < NN; i++) {
        float r = acc[i];
#pragma unroll
        for (int o = 16; o; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
        if (lane == 0 && r != 0.f) {
          const int jx = D3 ? i % NW : 0, jy = D3 ? (i / NW) % NW : i % NW, jz = D3 ? i / (NW * NW) : i / NW;
          const int gx = D3 ? c[0] + jx + J0 + gd.g[0] : 0;
          atomicAdd(&rho[((c[2] + jz + J0 + gd.g[2]) * gd.ext[1] + (c[1] + jy + J0 + gd.g[1])) * gd.ext[0] + gx], r);
        }
      }
    }
    // the records of this cell's exchange row: lane = record; each sits in a neighbouring cell
    const unsigned mine = lane < ND ? xin.mask[(size_t)k * XW + lane] : 0u;
    int dc = -1;
    for (int d = 0; d < ND; d++)
      if ((__shfl_sync(0xffffffffu, mine, d) >> lane) & 1u) dc = d;
    if (dc >= 0) {
      const XRec r = xin.rec[(size_t)k * PSC_XCAP + lane];
      int sx, sy, sz;
      dir_decode<D3>(dc, sx, sy, sz);
      const int cx = D3 ? wrap_cell(c[0] + sx, gd.n[0]) : 0, cy = wrap_cell(c[1] + sy, gd.n[1]),
                cz = wrap_cell(c[2] + sz, gd.n[2]);
      const float ax = __uint_as_float(r.a.x), ay = __uint_as_float(D3 ? r.a.y : r.a.x),
                  az = __uint_as_float(D3 ? r.a.z : r.a.y);
      const float q = __uint_as_float(D3 ? r.b.z : r.b.y) * gd.inv_dV;
      float wx[NW], wy[NW], wz[NW];
      if (D3) node_weights<ORDER>(ax, wx);
      node_weights<ORDER>(ay, wy);
      node_weights<ORDER>(az, wz);
      for (int jz = 0; jz < NW; jz++)
        for (int jy = 0; jy < NW; jy++)
          for (int jx = 0; jx < (D3 ? NW : 1); jx++) {
            const float v = q * wz[jz] * wy[jy] * (D3 ? wx[jx] : 1.f);
            if (v != 0.f)
              atomicAdd(&rho[((cz + jz + J0 + gd.g[2]) * gd.ext[1] + (cy + jy + J0 + gd.g[1])) * gd.ext[0] +
                             (D3 ? cx + jx + J0 + gd.g[0] : 0)], v);
          }
    }
  }
}

struct Pt3 {
  int c[3];
};
__device__ __forceinline__ Pt3 decode3(const GridDesc &gd, int idx) {
  Pt3 p;
  p.c[0] = idx % gd.ext[0];
  const int r = idx / gd.ext[0];
  p.c[1] = r % gd.ext[1];
  p.c[2] = r / gd.ext[1];
  return p;
}
// offsets to the +1 / -1 neighbour along d, wrapped periodically inside the extended array
__device__ __forceinline__ int up3(const GridDesc &gd, const Pt3 &p, int d) {
  return (p.c[d] + 1 < gd.ext[d]) ? gd.nbo[d] : -(gd.n[d] - 1) * gd.nbo[d];
}
__device__ __forceinline__ int down3(const GridDesc &gd, const Pt3 &p, int d) {
  return (p.c[d] > 0) ? -gd.nbo[d] : (gd.n[d] - 1) * gd.nbo[d];
}

// f = div- E - rho at every point of the extended array (a ghost point repeats the arithmetic of
// its periodic image on identical values)
__global__ void __launch_bounds__(MT)
k_gauss_residual(GridDesc gd, const float *__restrict__ E, const float *__restrict__ rho, float *__restrict__ f) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= gd.comp) return;
  const Pt3 p = decode3(gd, idx);
  const float *Ex = E, *Ey = E + gd.comp, *Ez = E + 2 * gd.comp;
  float d = 0.f;
  if (gd.n[0] > 1) d += (Ex[idx] - Ex[idx + down3(gd, p, 0)]) * gd.inv_dx[0];
  if (gd.n[1] > 1) d += (Ey[idx] - Ey[idx + down3(gd, p, 1)]) * gd.inv_dx[1];
  if (gd.n[2] > 1) d += (Ez[idx] - Ez[idx + down3(gd, p, 2)]) * gd.inv_dx[2];
  f[idx] = d - rho[idx];
}

// E += D grad+ f
__global__ void __launch_bounds__(MT)
k_marder_apply(GridDesc gd, float *__restrict__ E, const float *__restrict__ f, float D) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= gd.comp) return;
  const Pt3 p = decode3(gd, idx);
  const float f0 = f[idx];
  if (gd.n[0] > 1) E[idx] += D * (f[idx + up3(gd, p, 0)] - f0) * gd.inv_dx[0];
  if (gd.n[1] > 1) E[idx + gd.comp] += D * (f[idx + up3(gd, p, 1)] - f0) * gd.inv_dx[1];
  if (gd.n[2] > 1) E[idx + 2 * gd.comp] += D * (f[idx + up3(gd, p, 2)] - f0) * gd.inv_dx[2];
}

}  // namespace

// node charge density of the cell store into c->rho component 0 (ghosts folded and refilled)
int psc_charge_density_internal(psc_ctx *c, cudaStream_t s) {
  const GridDesc &gd = c->gd;
  if (!c->rho) {
    PSC_CUDA_TRY(c, cudaMalloc((void **)&c->rho, (size_t)3 * gd.comp * sizeof(float)));
  }
  PSC_CUDA_TRY(c, cudaMemsetAsync(c->rho, 0, (size_t)3 * gd.comp * sizeof(float), s));
  c->launches++;
  const Cols &in = c->cols[c->cur];
  const Exchange &xin = c->xch[c->xcur];
  const int blocks = (int)min((int64_t)c->sm_count * 16, max((int64_t)1, cdiv64(gd.nkeys, MT / 32)));
  const bool d3 = psc_is3d(gd);
  if (d3 && gd.order == 1) k_rho<true, 1><<<blocks, MT, 0, s>>>(gd, in, c->base, c->cnt, xin, c->rho);
  else if (d3) k_rho<true, 2><<<blocks, MT, 0, s>>>(gd, in, c->base, c->cnt, xin, c->rho);
  else if (gd.order == 1) k_rho<false, 1><<<blocks, MT, 0, s>>>(gd, in, c->base, c->cnt, xin, c->rho);
  else k_rho<false, 2><<<blocks, MT, 0, s>>>(gd, in, c->base, c->cnt, xin, c->rho);
  PSC_LAUNCH_CHECK(c);
  int rc = psc_fields_fold(c, c->rho, s);
  if (rc) return rc;
  return psc_fields_fill_ghosts(c, c->rho, s);
}

int psc_marder_pass(psc_ctx *c, float D, int iters, cudaStream_t s) {
  const GridDesc &gd = c->gd;
  int rc = psc_charge_density_internal(c, s);
  if (rc) return rc;
  float *f = c->rho + gd.comp;  // second component of the scratch field
  const int blocks = (int)cdiv64(gd.comp, MT);
  for (int it = 0; it < iters; it++) {
    k_gauss_residual<<<blocks, MT, 0, s>>>(gd, c->E, c->rho, f);
    PSC_LAUNCH_CHECK(c);
    k_marder_apply<<<blocks, MT, 0, s>>>(gd, c->E, f, D);
    PSC_LAUNCH_CHECK(c);
  }
  return PSC_OK;
}

// ---- psc_marder_static: the same correction for callers that must not allocate --------------------
//
// psc_marder keeps rho and f in a field the context cudaMalloc's on its first use.  Some users of
// this library cannot afford that call where they apply the correction: a time loop that runs while
// another host thread captures a CUDA graph in the global capture mode (cudaMalloc is prohibited
// there and breaks the capture), a loop in which the implicit device-wide synchronisation of
// cudaMalloc would stall every other stream, or a process whose own memory pool (PyTorch's caching
// allocator, say) has already taken all of the HBM, so that a raw cudaMalloc from inside a library
// fails.  For them the scratch lives in the array below, which is part of the library's device
// image: every GPU that loads libpsc_b200.so holds these 3.75 MiB from then until the process
// exits, whether psc_marder_static is ever called or not.
//
// In host code the identifier g_marder_scratch is only a handle of the symbol, not a device
// address (passing it to a kernel would make the kernel fault, or scribble over host memory on a
// system where the GPU can reach it), so the host asks the runtime for the address once per
// device, with that device current, and hands the kernels that pointer.
static __device__ __align__(256) float g_marder_scratch[3 * PSC_MARDER_STATIC_MAX_POINTS];

namespace {

constexpr int STATIC_MAX_DEVICES = 64;
float *g_marder_scratch_addr[STATIC_MAX_DEVICES];  // device address of the array on device i (0: not asked yet)
std::mutex g_marder_scratch_mu;

// Address of g_marder_scratch on the CURRENT device.  The first call on a device resolves the
// symbol (which may make the runtime load the module on that device); later calls read the table.
int marder_static_scratch(psc_ctx *c, float **out) {
  int dev = -1;
  PSC_CUDA_TRY(c, cudaGetDevice(&dev));
  if (dev < 0 || dev >= STATIC_MAX_DEVICES) return PSC_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_marder_scratch_mu);
  if (!g_marder_scratch_addr[dev]) {
    float *p = nullptr;
    PSC_CUDA_TRY(c, cudaGetSymbolAddress((void **)&p, g_marder_scratch));
    if (!p) return PSC_ERR_CUDA;
    g_marder_scratch_addr[dev] = p;
  }
  *out = g_marder_scratch_addr[dev];
  return PSC_OK;
}

}  // namespace

extern "C" int psc_marder_static(psc_ctx *c, void *stream, float diffusion, int iters) {
  if (!c || iters < 0 || !(diffusion >= 0.f)) return PSC_ERR_INVALID_ARG;
  if (!c->have_particles || !c->have_fields || !c->ws || c->ws_cap != c->np) return PSC_ERR_NOT_BOUND;
  if (c->state != PSC_STATE_STORE) return PSC_ERR_NOT_SORTED;
  const GridDesc &gd = c->gd;
  if ((int64_t)gd.comp > (int64_t)PSC_MARDER_STATIC_MAX_POINTS) return PSC_ERR_SCRATCH_LIMIT;
  double lap = 0.0;  // the same bound on the diffusion number as psc_marder
  for (int d = 0; d < 3; d++)
    if (gd.n[d] > 1) lap += 4.0 / ((double)gd.dx[d] * (double)gd.dx[d]);
  if ((double)diffusion * lap > 1.0 + 1e-6) return PSC_ERR_CFL;
  float *scratch = nullptr;
  int rc = marder_static_scratch(c, &scratch);
  if (rc) return rc;
  cudaStream_t s = (cudaStream_t)stream;
  if ((rc = psc_store_relayout_if_spilled(c, s))) return rc;  // nobody may be waiting in the spill list

  // The array still holds whatever the previous call (of any context on this device) left in it.
  // rho is accumulated with atomics and must start from zero; f is overwritten point by point
  // before it is read; the third component is only there because the ghost kernels work on three.
  float *rho = scratch, *f = scratch + gd.comp;
  PSC_CUDA_TRY(c, cudaMemsetAsync(scratch, 0, (size_t)3 * gd.comp * sizeof(float), s));
  c->launches++;
  const Cols &in = c->cols[c->cur];
  const Exchange &xin = c->xch[c->xcur];
  const int rblocks = (int)min((int64_t)c->sm_count * 16, max((int64_t)1, cdiv64(gd.nkeys, MT / 32)));
  const bool d3 = psc_is3d(gd);
  if (d3 && gd.order == 1) k_rho<true, 1><<<rblocks, MT, 0, s>>>(gd, in, c->base, c->cnt, xin, rho);
  else if (d3) k_rho<true, 2><<<rblocks, MT, 0, s>>>(gd, in, c->base, c->cnt, xin, rho);
  else if (gd.order == 1) k_rho<false, 1><<<rblocks, MT, 0, s>>>(gd, in, c->base, c->cnt, xin, rho);
  else k_rho<false, 2><<<rblocks, MT, 0, s>>>(gd, in, c->base, c->cnt, xin, rho);
  PSC_LAUNCH_CHECK(c);
  if ((rc = psc_fields_fold(c, scratch, s))) return rc;
  if ((rc = psc_fields_fill_ghosts(c, scratch, s))) return rc;
  const int blocks = (int)cdiv64(gd.comp, MT);
  for (int it = 0; it < iters; it++) {
    k_gauss_residual<<<blocks, MT, 0, s>>>(gd, c->E, rho, f);
    PSC_LAUNCH_CHECK(c);
    k_marder_apply<<<blocks, MT, 0, s>>>(gd, c->E, f, diffusion);
    PSC_LAUNCH_CHECK(c);
  }
  return PSC_OK;
}
