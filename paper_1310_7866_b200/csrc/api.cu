// api.cu -- the C ABI of include/psc.h: context, binding, the time step of Fig. 8.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include "psc_internal.cuh"

namespace {

// x may be NULL when x is the invariant direction of a 2-d run (then it is not carried)
bool cols_complete(const psc_ctx *ctx, const psc_particle_cols *c) {
  return (c->x || ctx->gd.n[0] == 1) && c->y && c->z && c->ux && c->uy && c->uz && c->qw && c->species;
}

Cols to_cols(const psc_particle_cols *c) {
  Cols o;
  o.x = c->x; o.y = c->y; o.z = c->z;
  o.ux = c->ux; o.uy = c->uy; o.uz = c->uz;
  o.qw = c->qw; o.sp = c->species; o.id = c->id;
  return o;
}

void prof_drain(psc_ctx *c, int ph) {
  Prof &pr = c->prof;
  const int n = pr.used[ph];
  if (n == 0) return;
  cudaEventSynchronize(pr.ev[ph][n - 1][1]);
  for (int i = 0; i < n; i++) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, pr.ev[ph][i][0], pr.ev[ph][i][1]) == cudaSuccess) {
      pr.ms[ph] += (double)ms;
      pr.cnt[ph]++;
    }
  }
  pr.used[ph] = 0;
}

}  // namespace

void psc_prof_begin(psc_ctx *c, int ph, cudaStream_t s) {
  Prof &pr = c->prof;
  if (!pr.on) return;
  if (pr.used[ph] == PSC_PROF_RING) prof_drain(c, ph);
  cudaEventRecord(pr.ev[ph][pr.used[ph]][0], s);
}

void psc_prof_end(psc_ctx *c, int ph, cudaStream_t s) {
  Prof &pr = c->prof;
  if (!pr.on) return;
  cudaEventRecord(pr.ev[ph][pr.used[ph]][1], s);
  pr.used[ph]++;
}

extern "C" {

const char *psc_version(void) { return "psc-b200 0.2 (sm_100a)"; }

const char *psc_strerror(int code) {
  switch (code) {
    case PSC_OK: return "ok";
    case PSC_ERR_INVALID_ARG: return "invalid argument";
    case PSC_ERR_NOT_BOUND: return "fields, particles or workspace not bound";
    case PSC_ERR_NOT_SORTED: return "particle list is not sorted";
    case PSC_ERR_CFL: return "time step too large (need dt <= min dx / 2)";
    case PSC_ERR_ALIGN: return "pointer not sufficiently aligned";
    case PSC_ERR_CUDA: return "CUDA runtime error (see psc_last_cuda_error)";
    case PSC_ERR_UNSUPPORTED: return "configuration not supported by this build";
    case PSC_ERR_WORKSPACE: return "workspace too small";
    case PSC_ERR_SCRATCH_LIMIT: return "grid larger than the fixed scratch array of psc_marder_static (PSC_MARDER_STATIC_MAX_POINTS)";
    default: return "unknown error";
  }
}

int psc_create(const psc_params *p, psc_ctx **out) {
  if (!p || !out) return PSC_ERR_INVALID_ARG;
  *out = nullptr;
  if (p->order != 1 && p->order != 2) return PSC_ERR_INVALID_ARG;
  if (p->scheme != PSC_SCHEME_STANDARD && p->scheme != PSC_SCHEME_ALTERNATING) return PSC_ERR_INVALID_ARG;
  if (p->n_species < 1 || p->n_species > PSC_MAX_SPECIES || !p->q || !p->m) return PSC_ERR_INVALID_ARG;
  if (p->ghost != PSC_GHOST) return PSC_ERR_INVALID_ARG;
  if (!(p->dt > 0.f)) return PSC_ERR_INVALID_ARG;
  int nact = 0;
  for (int d = 0; d < 3; d++) {
    if (p->n[d] != 1 && p->n[d] < 2 * PSC_GHOST) return PSC_ERR_INVALID_ARG;
    if (!(p->dx[d] > 0.f)) return PSC_ERR_INVALID_ARG;
    if (p->n[d] > 1) {
      nact++;
      if (p->dt > 0.5f * p->dx[d] * (1.f + 1e-6f)) return PSC_ERR_CFL;
    }
  }
  if (nact == 0) return PSC_ERR_INVALID_ARG;
  for (int s = 0; s < p->n_species; s++)
    if (!(p->m[s] > 0.f)) return PSC_ERR_INVALID_ARG;

  psc_ctx *c = (psc_ctx *)calloc(1, sizeof(psc_ctx));
  if (!c) return PSC_ERR_INVALID_ARG;
  GridDesc &gd = c->gd;
  const bool is3d = nact == 3;
  int64_t tot = 1, nk = 1;
  double dV = 1.0;
  for (int d = 0; d < 3; d++) {
    gd.n[d] = p->n[d];
    gd.g[d] = p->n[d] > 1 ? PSC_GHOST : 0;
    gd.ext[d] = gd.n[d] + 2 * gd.g[d];
    gd.dx[d] = p->dx[d];
    gd.inv_dx[d] = 1.0f / p->dx[d];
    gd.L[d] = (float)p->n[d] * p->dx[d];
    gd.dt_dx[d] = p->n[d] > 1 ? p->dt / p->dx[d] : 0.f;
    dV *= (double)p->dx[d];
    tot *= gd.ext[d];
    nk *= gd.n[d];
    int bs = p->block[d];
    if (p->n[d] == 1) bs = 1;
    if (bs == 0) {  // default supercell: 8x8 cells in 2-d, 4x4x4 in 3-d, shrunk to divide n
      bs = is3d ? 4 : 8;
      while (bs > 1 && p->n[d] % bs) bs >>= 1;
    }
    if (bs < 1 || p->n[d] % bs) {
      free(c);
      return PSC_ERR_INVALID_ARG;
    }
    gd.bs[d] = bs;
    gd.nb[d] = p->n[d] / bs;
  }
  // 32-bit indexing: 3 field components, and the exchange rows (32 records per cell)
  if (tot * 3 > 0x7fffffffLL || nk * PSC_XCAP > 0x7fffffffLL) {
    free(c);
    return PSC_ERR_INVALID_ARG;
  }
  gd.st[0] = 1;
  gd.st[1] = gd.ext[0];
  gd.st[2] = gd.ext[0] * gd.ext[1];
  for (int d = 0; d < 3; d++) gd.nbo[d] = gd.n[d] > 1 ? gd.st[d] : 0;
  gd.comp = (int)tot;
  gd.dt = p->dt;
  gd.inv_dV = (float)(1.0 / dV);
  for (int d = 0; d < 3; d++) gd.cur[d] = (float)((double)p->dx[d] / ((double)p->dt * dV));
  for (int d = 0; d < 3; d++) {
    gd.bsh[d] = -1;
    for (int k = 0; k < 12; k++)
      if (gd.bs[d] == (1 << k)) gd.bsh[d] = k;
  }
  gd.cpb = gd.bs[0] * gd.bs[1] * gd.bs[2];
  gd.nkeys = (int)nk;
  gd.ntiles = gd.nb[0] * gd.nb[1] * gd.nb[2];
  gd.order = p->order;
  gd.gmode = p->scheme;
  gd.nsp = p->n_species;
  gd.nd = is3d ? 27 : 9;
  for (int s = 0; s < p->n_species; s++) {
    c->q[s] = p->q[s];
    c->m[s] = p->m[s];
    gd.qmh[s] = (float)((double)p->q[s] * (double)p->dt / (2.0 * (double)p->m[s]));
  }
  // order 2 touches J nodes c-2..c+2 only while a particle moves less than half a cell
  // (A15): guaranteed by the dt check above.
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      cudaMalloc((void **)&c->d_flags, PSC_DW_COUNT * 4) != cudaSuccess ||
      cudaMemset(c->d_flags, 0, PSC_DW_COUNT * 4) != cudaSuccess) {
    c->last_err = (int)cudaGetLastError();
    if (c->d_flags) cudaFree(c->d_flags);
    free(c);
    return PSC_ERR_CUDA;  // no device: there is no CPU fallback
  }
  c->bufC = 64;
  *out = c;
  return PSC_OK;
}

void psc_destroy(psc_ctx *c) {
  if (!c) return;
  if (c->prof.have_events)
    for (int ph = 0; ph < PSC_PH_COUNT; ph++)
      for (int i = 0; i < PSC_PROF_RING; i++) {
        cudaEventDestroy(c->prof.ev[ph][i][0]);
        cudaEventDestroy(c->prof.ev[ph][i][1]);
      }
  if (c->d_flags) cudaFree(c->d_flags);
  if (c->rho) cudaFree(c->rho);
  free(c);
}

size_t psc_workspace_bytes(const psc_ctx *c, int64_t max_particles) {
  if (!c || max_particles < 0) return 0;
  return psc_sort_workspace_bytes(c, max_particles) + 256;
}

int psc_bind_workspace(psc_ctx *c, void *ws, size_t bytes) {
  if (!c || !ws) return PSC_ERR_INVALID_ARG;
  if (((uintptr_t)ws) & 255) return PSC_ERR_ALIGN;
  if (c->have_particles && c->form == PSC_FORM_REL) return PSC_ERR_INVALID_ARG;  // the store's tables live in ws
  c->ws = ws;
  c->ws_bytes = bytes;
  c->ws_cap = -1;
  c->have_sort_result = 0;
  if (c->have_particles) {
    if (bytes < psc_workspace_bytes(c, c->np)) return PSC_ERR_WORKSPACE;
    const int rc = psc_sort_carve(c, c->np);
    if (rc) return rc;
    c->ws_cap = c->np;
  }
  return PSC_OK;
}

int64_t psc_field_elems(const psc_ctx *c, int32_t ext[3]) {
  if (!c) return 0;
  if (ext)
    for (int d = 0; d < 3; d++) ext[d] = c->gd.ext[d];
  return 3 * (int64_t)c->gd.comp;
}

int psc_bind_fields(psc_ctx *c, float *E, float *B, float *J) {
  if (!c || !E || !B || !J) return PSC_ERR_INVALID_ARG;
  if ((((uintptr_t)E) | ((uintptr_t)B) | ((uintptr_t)J)) & 15) return PSC_ERR_ALIGN;
  c->E = E;
  c->B = B;
  c->J = J;
  c->have_fields = 1;
  psc_make_tile_maps(c);  // optional: the 3-d order-1 kernel stages its tiles by TMA where they apply
  return PSC_OK;
}

int64_t psc_particle_capacity(const psc_ctx *c, int64_t n) {
  if (!c || n < 0) return 0;
  return psc_store_capacity(c, n);
}

int psc_bind_particles(psc_ctx *c, int64_t n, int64_t capacity, const psc_particle_cols *a,
                       const psc_particle_cols *b) {
  if (!c || !a || !b || n < 0 || n > 0x6fffff00LL) return PSC_ERR_INVALID_ARG;
  if (!cols_complete(c, a) || !cols_complete(c, b)) return PSC_ERR_INVALID_ARG;
  if ((a->id == nullptr) != (b->id == nullptr)) return PSC_ERR_INVALID_ARG;
  if ((a->x == nullptr) != (b->x == nullptr)) return PSC_ERR_INVALID_ARG;
  if (capacity < psc_store_capacity(c, n)) return PSC_ERR_WORKSPACE;
  if (capacity > 0x7fffff00LL) return PSC_ERR_INVALID_ARG;  // 32-bit slot indices
  const void *ptrs[] = {a->x, a->y, a->z, a->ux, a->uy, a->uz, a->qw, a->species, a->id,
                        b->x, b->y, b->z, b->ux, b->uy, b->uz, b->qw, b->species, b->id};
  for (const void *p : ptrs)
    if (((uintptr_t)p) & 15) return PSC_ERR_ALIGN;
  c->cols[0] = to_cols(a);
  c->cols[1] = to_cols(b);
  c->cur = 0;
  c->np = n;
  c->capacity = capacity;
  c->have_particles = 1;
  c->state = PSC_STATE_UNSORTED;
  c->form = PSC_FORM_ABS;
  c->xcur = 0;
  c->have_sort_result = 0;
  if (c->ws) {
    if (c->ws_bytes < psc_workspace_bytes(c, n)) {
      c->ws_cap = -1;
      return PSC_ERR_WORKSPACE;
    }
    const int rc = psc_sort_carve(c, n);
    if (rc) return rc;
    c->ws_cap = n;
  }
  return PSC_OK;
}

int psc_particles_sort(psc_ctx *c, void *stream) {
  if (!c) return PSC_ERR_INVALID_ARG;
  if (!c->have_particles || !c->ws || c->ws_cap != c->np) return PSC_ERR_NOT_BOUND;
  cudaStream_t s = (cudaStream_t)stream;
  ProfScope ps(c, PSC_PH_SORT, s);
  return psc_sort_general(c, s);  // the physically sorted, stable list this call promises
}

// the sort as psc_step uses it: a store keeps itself ordered by cell; only a
// push that spilled makes the device lay it out again
static int sort_lazy(psc_ctx *c, cudaStream_t s) {
  if (!c->have_particles || !c->ws || c->ws_cap != c->np) return PSC_ERR_NOT_BOUND;
  ProfScope ps(c, PSC_PH_SORT, s);
  if (c->state == PSC_STATE_STORE) return psc_store_relayout_if_spilled(c, s);
  return psc_sort_general(c, s);
}

int psc_push_particles(psc_ctx *c, void *stream) {
  if (!c) return PSC_ERR_INVALID_ARG;
  if (!c->have_particles || !c->have_fields || !c->ws || c->ws_cap != c->np) return PSC_ERR_NOT_BOUND;
  if (c->state != PSC_STATE_STORE || c->form != PSC_FORM_REL) return PSC_ERR_NOT_SORTED;
  cudaStream_t s = (cudaStream_t)stream;
  if (!c->in_step) {  // (psc_step has just done this)
    ProfScope ps(c, PSC_PH_SORT, s);
    const int rc = psc_store_relayout_if_spilled(c, s);
    if (rc) return rc;
  }
  {
    ProfScope ps(c, PSC_PH_J_ZERO, s);
    PSC_CUDA_TRY(c, cudaMemsetAsync(c->J, 0, (size_t)3 * c->gd.comp * sizeof(float), s));
    c->launches++;
  }
  const int rc = c->gd.order == 1 ? psc_push_order1(c, s) : psc_push_order2(c, s);
  if (rc) return rc;
  c->xcur ^= 1;  // the leavers' records are in the exchange the next push reads
  c->have_sort_result = 0;
  return PSC_OK;
}

int psc_push_fields(psc_ctx *c, int which, float frac, void *stream) {
  if (!c || !(frac > 0.f)) return PSC_ERR_INVALID_ARG;
  if (!c->have_fields) return PSC_ERR_NOT_BOUND;
  if (which == PSC_B) {
    ProfScope ps(c, PSC_PH_FIELD_B, (cudaStream_t)stream);
    return psc_fields_push_b(c, frac, (cudaStream_t)stream);
  }
  if (which == PSC_E) {
    ProfScope ps(c, PSC_PH_FIELD_E, (cudaStream_t)stream);
    return psc_fields_push_e(c, frac, (cudaStream_t)stream);
  }
  return PSC_ERR_INVALID_ARG;
}

int psc_charge_density(psc_ctx *c, void *stream, float *rho) {
  if (!c || !rho) return PSC_ERR_INVALID_ARG;
  if (!c->have_particles || !c->ws || c->ws_cap != c->np) return PSC_ERR_NOT_BOUND;
  if (c->state != PSC_STATE_STORE) return PSC_ERR_NOT_SORTED;
  cudaStream_t s = (cudaStream_t)stream;
  int rc = psc_store_relayout_if_spilled(c, s);  // nobody may be waiting in the spill list
  if (rc) return rc;
  if ((rc = psc_charge_density_internal(c, s))) return rc;
  PSC_CUDA_TRY(c, cudaMemcpyAsync(rho, c->rho, (size_t)c->gd.comp * sizeof(float), cudaMemcpyDeviceToDevice, s));
  c->launches++;
  return PSC_OK;
}

int psc_patch_loads(psc_ctx *c, void *stream, const int32_t patch_blocks[3], int64_t *loads, int32_t np_out[3]) {
  if (!c || !patch_blocks || !loads) return PSC_ERR_INVALID_ARG;
  if (!c->have_particles || !c->ws || c->ws_cap != c->np) return PSC_ERR_NOT_BOUND;
  if (c->state != PSC_STATE_STORE) return PSC_ERR_NOT_SORTED;
  return psc_patch_loads_internal(c, (cudaStream_t)stream, patch_blocks, loads, np_out);
}

int psc_marder(psc_ctx *c, void *stream, float diffusion, int iters) {
  if (!c || iters < 0 || !(diffusion >= 0.f)) return PSC_ERR_INVALID_ARG;
  if (!c->have_particles || !c->have_fields || !c->ws || c->ws_cap != c->np) return PSC_ERR_NOT_BOUND;
  if (c->state != PSC_STATE_STORE) return PSC_ERR_NOT_SORTED;
  double lap = 0.0;  // largest eigenvalue of -div- grad+: sum 4/dx^2; a pass must not overshoot
  for (int d = 0; d < 3; d++)
    if (c->gd.n[d] > 1) lap += 4.0 / ((double)c->gd.dx[d] * (double)c->gd.dx[d]);
  if ((double)diffusion * lap > 1.0 + 1e-6) return PSC_ERR_CFL;
  cudaStream_t s = (cudaStream_t)stream;
  const int rc = psc_store_relayout_if_spilled(c, s);
  if (rc) return rc;
  ProfScope ps(c, PSC_PH_MARDER, s);
  return psc_marder_pass(c, diffusion, iters, s);
}

int psc_fill_ghosts(psc_ctx *c, int which, void *stream) {
  if (!c) return PSC_ERR_INVALID_ARG;
  if (!c->have_fields) return PSC_ERR_NOT_BOUND;
  float *F = which == PSC_E ? c->E : which == PSC_B ? c->B : which == PSC_J ? c->J : nullptr;
  if (!F) return PSC_ERR_INVALID_ARG;
  return psc_fields_fill_ghosts(c, F, (cudaStream_t)stream);
}

int psc_exchange_j(psc_ctx *c, void *stream) {
  if (!c) return PSC_ERR_INVALID_ARG;
  if (!c->have_fields) return PSC_ERR_NOT_BOUND;
  ProfScope ps(c, PSC_PH_J_EXCHANGE, (cudaStream_t)stream);
  int rc = psc_fields_fold(c, c->J, (cudaStream_t)stream);
  if (rc) return rc;
  return psc_fields_fill_ghosts(c, c->J, (cudaStream_t)stream);
}

// Fig. 8.  On one GPU the "single synchronisation point" is stream order:
// exchange_particles is the periodic wrap inside the push, fill_ghosts_B is part of the B
// update (ghost points are computed like their images), add_and_fill_ghosts_j is psc_exchange_j.
int psc_step(psc_ctx *c, void *stream) {
  int rc;
  if (!c) return PSC_ERR_INVALID_ARG;
  if ((rc = sort_lazy(c, (cudaStream_t)stream))) return rc;
  if ((rc = psc_push_fields(c, PSC_B, 0.5f, stream))) return rc;  // B^n -> B^{n+1/2}
  c->in_step = 1;
  rc = psc_push_particles(c, stream);                             // p, x, j^{n+1}
  c->in_step = 0;
  if (rc) return rc;
  if ((rc = psc_push_fields(c, PSC_B, 0.5f, stream))) return rc;  // B^{n+1/2} -> B^{n+1}
  if ((rc = psc_exchange_j(c, stream))) return rc;
  if ((rc = psc_push_fields(c, PSC_E, 1.0f, stream))) return rc;  // E^{n+1/2} -> E^{n+3/2}
  return PSC_OK;
}

int psc_step_host(psc_ctx *c, void *stream, int64_t n, const psc_particle_cols *h, float *hE,
                  float *hB, float *hJ, int nsteps) {
  if (!c || !h || !hE || !hB || nsteps < 0) return PSC_ERR_INVALID_ARG;
  if (!c->have_particles || !c->have_fields || !c->ws) return PSC_ERR_NOT_BOUND;
  if (n != c->np || !cols_complete(c, h)) return PSC_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  const size_t fb = (size_t)3 * c->gd.comp * 4, pb = (size_t)n * 4;
  {
    c->cur = 0;  // the dense set takes the host's particles; the sort below files them into the store set
    Cols &d = c->cols[c->cur];
    if ((d.id != nullptr) != (h->id != nullptr)) return PSC_ERR_INVALID_ARG;
    if ((d.x != nullptr) != (h->x != nullptr)) return PSC_ERR_INVALID_ARG;
    const void *src[] = {h->x, h->y, h->z, h->ux, h->uy, h->uz, h->qw, h->species, h->id};
    void *dst[] = {d.x, d.y, d.z, d.ux, d.uy, d.uz, d.qw, d.sp, d.id};
    for (int i = 0; i < 9; i++)
      if (dst[i]) PSC_CUDA_TRY(c, cudaMemcpyAsync(dst[i], src[i], pb, cudaMemcpyHostToDevice, s));
    PSC_CUDA_TRY(c, cudaMemcpyAsync(c->E, hE, fb, cudaMemcpyHostToDevice, s));
    PSC_CUDA_TRY(c, cudaMemcpyAsync(c->B, hB, fb, cudaMemcpyHostToDevice, s));
    c->state = PSC_STATE_UNSORTED;
    c->form = PSC_FORM_ABS;
    c->have_sort_result = 0;
    c->launches += 11;
  }
  for (int i = 0; i < nsteps; i++) {
    const int rc = psc_step(c, stream);
    if (rc) return rc;
  }
  {
    const int rc = psc_particles_export(c, stream);
    if (rc) return rc;
    Cols &d = c->cols[c->cur];
    void *dst[] = {h->x, h->y, h->z, h->ux, h->uy, h->uz, h->qw, h->species, h->id};
    const void *src[] = {d.x, d.y, d.z, d.ux, d.uy, d.uz, d.qw, d.sp, d.id};
    for (int i = 0; i < 9; i++)
      if (src[i]) PSC_CUDA_TRY(c, cudaMemcpyAsync(dst[i], src[i], pb, cudaMemcpyDeviceToHost, s));
    PSC_CUDA_TRY(c, cudaMemcpyAsync(hE, c->E, fb, cudaMemcpyDeviceToHost, s));
    PSC_CUDA_TRY(c, cudaMemcpyAsync(hB, c->B, fb, cudaMemcpyDeviceToHost, s));
    if (hJ) PSC_CUDA_TRY(c, cudaMemcpyAsync(hJ, c->J, fb, cudaMemcpyDeviceToHost, s));
    c->launches += 12;
  }
  PSC_CUDA_TRY(c, cudaStreamSynchronize(s));
  return PSC_OK;
}

int psc_sort_result(psc_ctx *c, void *stream, const int32_t **cell_idx, const int32_t **perm,
                    const int32_t **cell_offsets, int64_t *n_keys) {
  if (!c) return PSC_ERR_INVALID_ARG;
  if (!c->have_sort_result) return PSC_ERR_NOT_SORTED;
  if (cell_idx) {
    const int rc = psc_sort_cell_idx(c, (cudaStream_t)stream);
    if (rc) return rc;
    *cell_idx = c->cell_idx;
  }
  if (perm) *perm = c->perm;
  if (cell_offsets) *cell_offsets = c->offs_dense;
  if (n_keys) *n_keys = c->gd.nkeys;
  return PSC_OK;
}

int psc_particles_form(const psc_ctx *c) { return c ? c->form : PSC_ERR_INVALID_ARG; }

int psc_particles_gather(psc_ctx *c, void *stream, const psc_particle_cols *dst, int32_t *key,
                         int absolute) {
  if (!c || !dst) return PSC_ERR_INVALID_ARG;
  if (!c->have_particles || !c->ws || c->ws_cap != c->np) return PSC_ERR_NOT_BOUND;
  if (c->form != PSC_FORM_REL) return PSC_ERR_NOT_SORTED;
  if (!dst->y || !dst->z || !dst->ux || !dst->uy || !dst->uz || !dst->qw || !dst->species)
    return PSC_ERR_INVALID_ARG;
  return psc_store_gather(c, to_cols(dst), key, absolute != 0, (cudaStream_t)stream);
}

int psc_particles_export(psc_ctx *c, void *stream) {
  if (!c) return PSC_ERR_INVALID_ARG;
  if (!c->have_particles) return PSC_ERR_NOT_BOUND;
  if (c->form == PSC_FORM_ABS) return PSC_OK;
  if (!c->ws || c->ws_cap != c->np) return PSC_ERR_NOT_BOUND;
  const int rc = psc_store_gather(c, c->cols[c->cur ^ 1], nullptr, true, (cudaStream_t)stream);
  if (rc) return rc;
  c->cur ^= 1;
  c->form = PSC_FORM_ABS;
  c->state = PSC_STATE_UNSORTED;
  c->have_sort_result = 0;
  return PSC_OK;
}

int psc_particles_current(const psc_ctx *c, psc_particle_cols *out) {
  if (!c || !out) return PSC_ERR_INVALID_ARG;
  if (!c->have_particles) return PSC_ERR_NOT_BOUND;
  const Cols &d = c->cols[c->cur];
  out->x = d.x; out->y = d.y; out->z = d.z;
  out->ux = d.ux; out->uy = d.uy; out->uz = d.uz;
  out->qw = d.qw; out->species = d.sp; out->id = d.id;
  return PSC_OK;
}

int psc_store_info(psc_ctx *c, void *stream, int64_t info[8]) {
  if (!c || !info) return PSC_ERR_INVALID_ARG;
  uint32_t dw[PSC_DW_COUNT];
  PSC_CUDA_TRY(c, cudaMemcpyAsync(dw, c->d_flags, sizeof(dw), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  PSC_CUDA_TRY(c, cudaStreamSynchronize((cudaStream_t)stream));
  for (int i = 0; i < 8; i++) info[i] = 0;
  if (c->state == PSC_STATE_STORE) psc_refresh_image_size(c, dw);
  info[0] = dw[PSC_DW_MAXCNT];
  info[1] = dw[PSC_DW_SLOTS];
  info[2] = dw[PSC_DW_RELAYOUTS];
  info[3] = dw[PSC_DW_SPILL];
  info[4] = c->bufC;
  info[5] = c->used_tma;
  info[6] = dw[PSC_DW_INSERTED];
  return PSC_OK;
}

int psc_status(psc_ctx *c, void *stream, uint32_t *flags) {
  if (!c || !flags) return PSC_ERR_INVALID_ARG;
  uint32_t dw[PSC_DW_COUNT];
  PSC_CUDA_TRY(c, cudaMemcpyAsync(dw, c->d_flags, sizeof(dw), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  PSC_CUDA_TRY(c, cudaStreamSynchronize((cudaStream_t)stream));
  *flags = dw[PSC_DW_FLAGS];
  if (c->state == PSC_STATE_STORE) psc_refresh_image_size(c, dw);  // (the host has the block anyway)
  return PSC_OK;
}

int psc_profile(psc_ctx *c, void *stream, double *ms, int64_t *count) {
  if (!c || !ms || !count) return PSC_ERR_INVALID_ARG;
  PSC_CUDA_TRY(c, cudaStreamSynchronize((cudaStream_t)stream));
  for (int ph = 0; ph < PSC_PH_COUNT; ph++) {
    prof_drain(c, ph);
    ms[ph] = c->prof.ms[ph];
    count[ph] = c->prof.cnt[ph];
    c->prof.ms[ph] = 0.0;
    c->prof.cnt[ph] = 0;
  }
  return PSC_OK;
}

int64_t psc_launch_count(const psc_ctx *c) { return c ? c->launches : 0; }
int psc_last_cuda_error(const psc_ctx *c) { return c ? c->last_err : 0; }

int psc_set_option(psc_ctx *c, const char *name, int64_t value) {
  if (!c || !name) return PSC_ERR_INVALID_ARG;
  if (!strcmp(name, "profile")) {
    Prof &pr = c->prof;
    if (value && !pr.have_events) {
      for (int ph = 0; ph < PSC_PH_COUNT; ph++)
        for (int i = 0; i < PSC_PROF_RING; i++)
          for (int k = 0; k < 2; k++)
            if (cudaEventCreate(&pr.ev[ph][i][k]) != cudaSuccess) return PSC_ERR_CUDA;
      pr.have_events = 1;
    }
    if (!value)
      for (int ph = 0; ph < PSC_PH_COUNT; ph++) prof_drain(c, ph);
    pr.on = value != 0;
  } else if (!strcmp(name, "clear_flags")) {
    if (cudaMemset(c->d_flags, 0, 4) != cudaSuccess) return PSC_ERR_CUDA;
  } else return PSC_ERR_INVALID_ARG;
  return PSC_OK;
}

}  // extern "C"
