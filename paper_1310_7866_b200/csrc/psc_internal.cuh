// psc_internal.cuh -- internal declarations of the B200 PIC hot path (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "psc.h"

// Geometry + constants handed to every kernel by value (kernel-parameter space, broadcast
// through the constant bank).
struct GridDesc {
  int n[3];        // interior cells
  int g[3];        // ghost layers per direction (0 along an invariant direction)
  int ext[3];      // n + 2g
  int st[3];       // element strides of one component: {1, ext0, ext0*ext1}
  int nbo[3];      // neighbour offset per direction: st[d], or 0 along an invariant direction
  int comp;        // component stride ext0*ext1*ext2
  float dx[3], inv_dx[3], L[3];
  float dt;
  float dt_dx[3];    // dt / dx[d]  (0 along an invariant direction)
  float cur[3];      // dx[d] / (dt * dV): factor of the in-plane VB / Esirkepov current
  float inv_dV;
  int bs[3], nb[3];  // sort block (supercell) size in cells and number of blocks
  int cpb;           // cells per block
  int nkeys;         // total cells
  int ntiles;        // number of blocks
  int order;
  int nsp;
  int nd;            // direction codes of a move: 9 (2-d) or 27 (3-d); see dir_code()
  float qmh[PSC_MAX_SPECIES];  // q_s dt / (2 m_s), the Boris h
};

struct Cols {
  float *x, *y, *z, *ux, *uy, *uz, *qw;
  int32_t *sp;
  int32_t *id;
};

// Where the particle list is in the sort / push cycle (internal form unless UNSORTED):
//   UNSORTED  absolute positions in arbitrary order (after bind or export)
//   SORTED    the current column set is physically in sorted order; offs[ocur] = cell offsets
//   PUSHED    the current set is the list a push wrote: cell k's particles of BEFORE the push in
//             [offs[ocur][k], offs[ocur][k+1]), its stayers first (dircnt[STAY][k] of them), then
//             its leavers, each leaver with the direction code of its move in dcode[slot];
//             dircnt holds the per-cell code counts
//   INDEXED   the current set is still that written list (layout offs[ocur^1]); offs[ocur] are
//             the cell offsets of the new order, nstay / aoffs / alist say where each cell's
//             particles are (a run of stayers + listed arrivals; reorder happens on the next
//             load); dircnt[dc != STAY][k] now hold arrival-list bases
enum { PSC_STATE_UNSORTED = 0, PSC_STATE_SORTED = 1, PSC_STATE_PUSHED = 2, PSC_STATE_INDEXED = 3 };
enum { PSC_FORM_ABS = 0, PSC_FORM_REL = 1 };

// Direction code of a move by (sx, sy, sz) in {-1,0,1}^3 cells (a particle moves at
// most one cell per step, so 9 (2-d) / 27 (3-d) destination classes exist).  2-d (yz plane):
// (sy+1) + 3 (sz+1), "stay" = 4; 3-d: (sx+1) + 3 (sy+1) + 9 (sz+1), "stay" = 13.
template <bool D3>
__host__ __device__ __forceinline__ int dir_code(int sx, int sy, int sz) {
  return D3 ? (sx + 1) + 3 * (sy + 1) + 9 * (sz + 1) : (sy + 1) + 3 * (sz + 1);
}

// per-phase CUDA-event timing (psc_profile): a ring of start/stop pairs per phase
constexpr int PSC_PROF_RING = 64;
struct Prof {
  int on;
  int have_events;
  cudaEvent_t ev[PSC_PH_COUNT][PSC_PROF_RING][2];
  int used[PSC_PH_COUNT];
  double ms[PSC_PH_COUNT];
  int64_t cnt[PSC_PH_COUNT];
};

struct psc_ctx {
  GridDesc gd;
  Prof prof;
  float q[PSC_MAX_SPECIES], m[PSC_MAX_SPECIES];
  float *E, *B, *J;
  Cols cols[2];
  int cur;
  int64_t np;
  int have_particles, have_fields;
  int state;
  int form;        // PSC_FORM_ABS: absolute positions; PSC_FORM_REL: in-cell offsets
  int ocur;        // offs[ocur]: offsets of the latest sort
  int have_sort_result;  // 0: none; 1: key[] holds the input keys of the last general sort
  // workspace carve-up (all device pointers)
  void *ws;
  size_t ws_bytes;
  int64_t ws_cap;  // max particles the bound workspace was sized for
  int32_t *key, *curkey, *perm, *cell_idx, *offs[2], *cursor, *big_list, *dircnt;
  int32_t *alist, *aoffs, *nstay;  // index sort: arrival list, its per-cell offsets, stayers per cell
  long long *pack, *packloc, *scan_tmp;
  uint8_t *dcode;
  uint32_t *d_flags;  // owned: 16 words; [0] sticky flags, [1] big-segment counter
  int64_t launches;
  int last_err;
  int sm_count;
  // options
  int opt_push_variant;  // 0: default; 1: 2-d default tile at 6 blocks/SM; 2: run-time tile geometry
  int opt_threads;       // threads per block of the particle kernels (0: default)
};

#define PSC_CUDA_TRY(ctx, expr)                   \
  do {                                            \
    cudaError_t e__ = (expr);                     \
    if (e__ != cudaSuccess) {                     \
      (ctx)->last_err = (int)e__;                 \
      return PSC_ERR_CUDA;                        \
    }                                             \
  } while (0)

#define PSC_LAUNCH_CHECK(ctx)                     \
  do {                                            \
    (ctx)->launches++;                            \
    cudaError_t e__ = cudaGetLastError();         \
    if (e__ != cudaSuccess) {                     \
      (ctx)->last_err = (int)e__;                 \
      return PSC_ERR_CUDA;                        \
    }                                             \
  } while (0)

static inline int64_t cdiv64(int64_t a, int64_t b) { return (a + b - 1) / b; }

// api.cu: phase brackets (no-ops unless profiling is on)
void psc_prof_begin(psc_ctx *c, int phase, cudaStream_t s);
void psc_prof_end(psc_ctx *c, int phase, cudaStream_t s);
struct ProfScope {
  psc_ctx *c; int ph; cudaStream_t s;
  ProfScope(psc_ctx *c_, int ph_, cudaStream_t s_) : c(c_), ph(ph_), s(s_) { psc_prof_begin(c, ph, s); }
  ~ProfScope() { psc_prof_end(c, ph, s); }
};

// fields.cu
int psc_fields_push_b(psc_ctx *c, float frac, cudaStream_t s);
int psc_fields_push_e(psc_ctx *c, float frac, cudaStream_t s);
int psc_fields_fill_ghosts(psc_ctx *c, float *F, cudaStream_t s);
int psc_fields_fold(psc_ctx *c, float *F, cudaStream_t s);
// sort.cu
size_t psc_sort_workspace_bytes(const psc_ctx *c, int64_t n);
int psc_sort_carve(psc_ctx *c, int64_t n);
int psc_sort_general(psc_ctx *c, cudaStream_t s);      // any state -> SORTED (stable)
int psc_sort_index(psc_ctx *c, cudaStream_t s);        // PUSHED -> INDEXED
int psc_sort_cell_idx(psc_ctx *c, cudaStream_t s);
int psc_sort_current_keys(psc_ctx *c, cudaStream_t s);  // key[] := keys of the current particles
int psc_particles_to_abs(psc_ctx *c, cudaStream_t s);
// push1.cu / push2.cu
int psc_push_order1(psc_ctx *c, cudaStream_t s);
int psc_push_order2(psc_ctx *c, cudaStream_t s);
