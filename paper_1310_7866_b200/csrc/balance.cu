// balance.cu -- patch-based load balancing along a space-filling curve (PAPER.md:297-335,
// Appendix A).
//
// "Given a number of processing elements, decompose the domain into many more patches than there
// are processing elements ... By dynamically shifting the assignment of patches to processing
// elements we can ensure that each processing element is assigned a nearly equal load"
// (PAPER.md:301).  Three parts:
//   * psc_patch_loads   (device)  load of a patch = its particles + its cells, read
//                       off the cell store's per-cell counts and exchange-row headers: O(cells),
//                       no pass over the particles;
//   * psc_hilbert_order (host)    the Hilbert-Peano enumeration of the patches,
//                       by Skilling's transpose algorithm (bit manipulation on the curve index);
//   * psc_balance       (host)    Appendix A: cut the curve into one segment per rank so that each
//                       rank's load is closest to its share T_hat * C_r of the total.
#include <vector>

#include "store.cuh"

namespace {

struct PatchGeom {
  int pb[3];  // sort blocks per patch
  int np[3];  // patches
};

__device__ __forceinline__ int patch_of_cell(const GridDesc &gd, const PatchGeom &pg, const int c[3]) {
  const int p0 = (c[0] / gd.bs[0]) / pg.pb[0], p1 = (c[1] / gd.bs[1]) / pg.pb[1], p2 = (c[2] / gd.bs[2]) / pg.pb[2];
  return (p2 * pg.np[1] + p1) * pg.np[0] + p0;
}

__global__ void __launch_bounds__(256)
k_patch_init(int npatch, long long cells_per_patch, unsigned long long *__restrict__ loads) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < npatch) loads[i] = (unsigned long long)cells_per_patch;
}

// a thread per cell: its residents count for the cell's patch, the records waiting in its
// exchange row for the patch of the cell they move to (one of 9 / 27 neighbours)
template <bool D3>
__global__ void __launch_bounds__(256)
k_patch_loads(GridDesc gd, PatchGeom pg, const int *__restrict__ cnt, const uint32_t *__restrict__ mask,
              unsigned long long *__restrict__ loads) {
  constexpr int XW = D3 ? PSC_XW3 : PSC_XW2, ND = D3 ? 27 : 9, STAY = D3 ? 13 : 4;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= gd.nkeys) return;
  int c[3];
  key_to_cell(gd, k, c);
  const int n = cnt[k];
  if (n) atomicAdd(&loads[patch_of_cell(gd, pg, c)], (unsigned long long)n);
  for (int dc = 0; dc < ND; dc++) {
    if (dc == STAY) continue;
    const int m = __popc(mask[(size_t)k * XW + dc]);
    if (!m) continue;
    int sx, sy, sz;
    dir_decode<D3>(dc, sx, sy, sz);
    const int d[3] = {D3 ? wrap_cell(c[0] + sx, gd.n[0]) : 0, wrap_cell(c[1] + sy, gd.n[1]),
                      wrap_cell(c[2] + sz, gd.n[2])};
    atomicAdd(&loads[patch_of_cell(gd, pg, d)], (unsigned long long)m);
  }
}

// the spill list: particles waiting for the next re-layout, filed under their destination key
__global__ void __launch_bounds__(256)
k_patch_spill(GridDesc gd, PatchGeom pg, const int *__restrict__ count, int cap, const int *__restrict__ key,
              unsigned long long *__restrict__ loads) {
  const int ns = min(*count, cap);
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < ns; i += gridDim.x * blockDim.x) {
    int c[3];
    key_to_cell(gd, key[i], c);
    atomicAdd(&loads[patch_of_cell(gd, pg, c)], 1ull);
  }
}

}  // namespace

int psc_patch_loads_internal(psc_ctx *c, cudaStream_t s, const int32_t pb[3], int64_t *loads, int32_t np_out[3]) {
  const GridDesc &gd = c->gd;
  PatchGeom pg;
  long long cells = 1;
  for (int d = 0; d < 3; d++) {
    if (pb[d] < 1 || gd.nb[d] % pb[d] != 0) return PSC_ERR_INVALID_ARG;
    pg.pb[d] = pb[d];
    pg.np[d] = gd.nb[d] / pb[d];
    cells *= (long long)pb[d] * gd.bs[d];
    if (np_out) np_out[d] = pg.np[d];
  }
  const int npatch = pg.np[0] * pg.np[1] * pg.np[2];
  unsigned long long *L = reinterpret_cast<unsigned long long *>(loads);
  k_patch_init<<<(npatch + 255) / 256, 256, 0, s>>>(npatch, cells, L);
  PSC_LAUNCH_CHECK(c);
  const uint32_t *mask = c->xch[c->xcur].mask;  // the rows the last push filled
  const int blocks = (gd.nkeys + 255) / 256;
  if (psc_is3d(gd)) k_patch_loads<true><<<blocks, 256, 0, s>>>(gd, pg, c->cnt, mask, L);
  else k_patch_loads<false><<<blocks, 256, 0, s>>>(gd, pg, c->cnt, mask, L);
  PSC_LAUNCH_CHECK(c);
  k_patch_spill<<<64, 256, 0, s>>>(gd, pg, c->spill.count, c->spill.cap, c->spill.key, L);
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}

// ---- Hilbert-Peano order (host) -------------------------------------------------------------
// Skilling's transpose form: the b*n-bit curve index h is spread over n words X[0..n) of b bits
// (bit j of X[i] = bit j*n + (n-1-i) of h); TransposeToAxes turns it into coordinates with a Gray
// decode followed by "undoing the excess work" (exchanges and inversions of low bits).
static void hilbert_axes(uint32_t *X, int b, int n) {
  const uint32_t N = 2u << (b - 1);
  uint32_t t = X[n - 1] >> 1;
  for (int i = n - 1; i > 0; i--) X[i] ^= X[i - 1];
  X[0] ^= t;
  for (uint32_t Q = 2; Q != N; Q <<= 1) {
    const uint32_t P = Q - 1;
    for (int i = n - 1; i >= 0; i--) {
      if (X[i] & Q) {
        X[0] ^= P;
      } else {
        t = (X[0] ^ X[i]) & P;
        X[0] ^= t;
        X[i] ^= t;
      }
    }
  }
}

extern "C" int psc_hilbert_order(const int32_t np[3], int32_t *order) {
  if (!np || !order) return PSC_ERR_INVALID_ARG;
  int act[3], n = 0, mx = 1;
  for (int d = 0; d < 3; d++) {
    if (np[d] < 1) return PSC_ERR_INVALID_ARG;
    if (np[d] > 1) act[n++] = d;
    if (np[d] > mx) mx = np[d];
  }
  if ((int64_t)np[0] * np[1] * np[2] > (int64_t)1 << 30) return PSC_ERR_INVALID_ARG;
  if (n == 0) {
    order[0] = 0;
    return PSC_OK;
  }
  int b = 0;
  while ((1 << b) < mx) b++;
  // the walk below visits every point of the enclosing cube: a very anisotropic grid such as
  // 2 x 2 x 65536 would need 2^48 of them (and 1 << 64 is undefined): refused
  if (b * n > 32) return PSC_ERR_UNSUPPORTED;
  const uint64_t total = (uint64_t)1 << (b * n);
  int64_t out = 0;
  for (uint64_t h = 0; h < total; h++) {
    uint32_t X[3] = {0, 0, 0};
    for (int j = 0; j < b; j++)
      for (int i = 0; i < n; i++)
        if ((h >> (j * n + (n - 1 - i))) & 1u) X[i] |= 1u << j;
    hilbert_axes(X, b, n);
    int p[3] = {0, 0, 0};
    bool inside = true;
    for (int i = 0; i < n; i++) {
      p[act[i]] = (int)X[i];
      inside = inside && (int)X[i] < np[act[i]];
    }
    if (inside) order[out++] = (p[2] * np[1] + p[1]) * np[0] + p[0];
  }
  return PSC_OK;
}

// ---- Appendix A (host) ------------------------------------------------------------------------
// Walk along the curve; a rank's segment [first, p] is closed when its load passes the rank's
// target T_hat * C_r (or when only as many patches as ranks are left): at the patch that crosses
// the target if that leaves the load closer to the target, else one patch earlier.
extern "C" int psc_balance(int64_t n_patches, const double *loads, int32_t n_ranks, const double *capability,
                           int32_t *count) {
  if (!loads || !capability || !count || n_ranks < 1 || n_patches < n_ranks) return PSC_ERR_INVALID_ARG;
  double l_total = 0.0, c_total = 0.0;
  for (int64_t p = 0; p < n_patches; p++) {
    if (!(loads[p] >= 0.0)) return PSC_ERR_INVALID_ARG;
    l_total += loads[p];
  }
  for (int r = 0; r < n_ranks; r++) {
    if (!(capability[r] > 0.0)) return PSC_ERR_INVALID_ARG;
    c_total += capability[r];
    count[r] = 0;
  }
  const double t_hat = l_total / c_total;  // target load per unit capability
  int r = 0;
  int64_t first = 0;   // first patch of rank r's segment
  double seg = 0.0;    // load of patches first .. p
  for (int64_t p = 0; p < n_patches && r < n_ranks - 1; p++) {
    seg += loads[p];
    const double target = t_hat * capability[r];
    const bool forced = (int64_t)(n_ranks - r) >= n_patches - p;  // as many ranks as patches left
    if (!(seg > target) && !forced) continue;
    const double above = seg - target, below = target - (seg - loads[p]);
    if (above > below && p > first) {  // closer without patch p: it opens the next rank's segment
      count[r] = (int32_t)(p - first);
      first = p;
      seg = loads[p];
    } else {
      count[r] = (int32_t)(p - first + 1);
      first = p + 1;
      seg = 0.0;
    }
    r++;
  }
  count[n_ranks - 1] = (int32_t)(n_patches - first);  // the last rank takes what is left
  return PSC_OK;
}

extern "C" int psc_balance_owners(int64_t n_patches, int32_t n_ranks, const int32_t *count, int32_t *owner) {
  if (!count || !owner || n_ranks < 1 || n_patches < 0) return PSC_ERR_INVALID_ARG;
  int64_t total = 0;
  for (int r = 0; r < n_ranks; r++) {
    if (count[r] < 0) return PSC_ERR_INVALID_ARG;
    total += count[r];
  }
  if (total != n_patches) return PSC_ERR_INVALID_ARG;
  int64_t i = 0;
  for (int r = 0; r < n_ranks; r++)
    for (int k = 0; k < count[r]; k++) owner[i++] = r;
  return PSC_OK;
}
