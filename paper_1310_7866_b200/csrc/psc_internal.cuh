// psc_internal.cuh -- internal declarations of the B200 PIC hot path (not part of the C ABI).
#pragma once
#include <cuda.h>  // CUtensorMap (type only: the encoder is fetched from the driver at run time)
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
  int bsh[3];        // log2 of bs[d] if it is a power of two, else -1 (cell_key without divisions)
  int cpb;           // cells per block
  int nkeys;         // total cells
  int ntiles;        // number of blocks
  int order;
  int nsp;
  int nd;            // direction codes of a move: 9 (2-d) or 27 (3-d); see dir_code()
  float qmh[PSC_MAX_SPECIES];  // q_s dt / (2 m_s), the Boris h
  int gmode;         // gather/deposit pairing (psc.h PSC_SCHEME_*)
};

struct Cols {
  float *x, *y, *z, *ux, *uy, *uz, *qw;
  int32_t *sp;
  int32_t *id;
};

// ---- the cell store -------------------------------------------------------
// In the internal form the particles of cell k (key order: block-major, cell-minor)
// are the slots [base[k], base[k] + cnt[k]) of the current column set.  base[] is fixed between
// layouts, a multiple of 32 slots (128 bytes per column), and leaves every cell spare capacity
// cap[k] = base[k+1] - base[k] >= cnt[k].  A push updates the particles that stay in their cell IN
// PLACE; a particle that leaves (at most one cell per direction and step) is written
// as a 32-byte record into the exchange rows of its SOURCE cell, tagged with the direction code of
// its move; the next push of the destination cell collects the records aimed at it from its 8 / 26
// neighbours' rows (reorder on load) and files them into the holes the cell's own
// leavers left.  So no per-step sort pass exists at all; the exchange is ping-pong buffered.
constexpr int PSC_XCAP = 32;        // exchange records per cell and step (one bit each in a header word)
constexpr int PSC_XW2 = 16, PSC_XW3 = 32;  // header words per row (2-d: 9 direction codes, 3-d: 27)
constexpr int PSC_SLOT_ALIGN = 32;  // cell segments start on multiples of 32 slots

// One exchange record: the first 8 buffer columns of a particle (see StoreDesc::col), positions
// relative to the DESTINATION cell.  2-d: {y z ux uy uz qw sp x2d}, 3-d: {x y z ux uy uz qw sp}.
struct __align__(16) XRec {
  uint4 a, b;
};

struct Exchange {
  XRec *rec;       // [nkeys * PSC_XCAP]
  uint32_t *mask;  // [nkeys * XW] row headers: mask[k * XW + dc] bit i <=> record i of row k moved by code dc
  int32_t *id;     // [nkeys * PSC_XCAP] or nullptr
};

// particles that found no room (exchange row or destination cell full): the next step re-lays
// the store out before it pushes (sort.cu: relayout)
struct Spill {
  XRec *rec;
  int32_t *key;   // destination cell
  int32_t *id;    // or nullptr
  int32_t *count; // device counter
  int cap;
};

// What a particle kernel reads and writes.  Column order of the per-warp shared-memory image of
// a cell ("buffer columns"): the DYNAMIC columns first (2-d: y z ux uy uz; 3-d: x y z ux uy uz),
// then the STATIC ones (qw, species, [carried x of a 2-d run], [id]).
struct StoreDesc {
  float *col[10];
  int ncol;        // buffer columns in use
  int ndyn;        // 5 or 6
  int icol_id;     // buffer column of id, or -1
  int icol_x2d;    // buffer column of the carried invariant coordinate, or -1
  const int32_t *base;
  int32_t *cnt;
  Exchange xin, xout;
  Spill spill;
  int imgC;        // slots of the per-warp cell image (multiple of 32, <= 256)
  int32_t *bigflag;  // [ntiles]: the image launch left a cell of this tile to the BIG launch
  uint8_t *bigcell;  // [nkeys]: ... this cell (set by the image launch, cleared by the BIG launch)
  uint32_t *nbig;    // tiles flagged by this step's image launch (the BIG launch returns at once if 0)
  uint32_t *nbig_next;  // the other step parity's counter: zeroed by this step's BIG launch
  uint32_t *flags;
  uint32_t *maxcnt;  // device word PSC_DW_MAXCNT: largest cell count (layouts, and cells that grew since)
  int maxcnt_known;  // its value when the host last read the status block: only a larger cell reports
};

// Where the particle list is in the sort / push cycle:
//   UNSORTED  absolute positions, dense [0, n), arbitrary order (after bind or export)
//   STORE     internal form: the cell store above (after psc_particles_sort, after a push)
enum { PSC_STATE_UNSORTED = 0, PSC_STATE_STORE = 1 };
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

// device status block (owned by the context): words
enum {
  PSC_DW_FLAGS = 0,    // sticky flags (psc_status)
  PSC_DW_BIG = 1,      // big-segment counter of the general sort
  PSC_DW_SPILL = 2,    // spill counter: != 0 => the next step re-lays the store out
  PSC_DW_MAXCNT = 3,   // largest cell count: of the last layout, raised by cells that grew since
  PSC_DW_SLOTS = 4,    // slots used by the last layout
  PSC_DW_RELAYOUTS = 5,  // number of re-layouts performed
  PSC_DW_NBIG = 6,     // [2]: tiles with a cell left to the BIG launch, by step parity
  PSC_DW_INSERTED = 8, // spilled particles filed straight into their cell (no re-layout needed), cumulative
  PSC_DW_COUNT = 16
};

// TMA tensor maps of the three field arrays (float[3][ez][ey][ex] as a 4-d tensor x, y, z,
// component) for the tile loads / the J-tile reduction of the 3-d order-1 kernel (push1.cu)
struct TileMaps {
  CUtensorMap E, B, J;
};

struct psc_ctx {
  GridDesc gd;
  TileMaps tmaps;
  int have_tmaps;  // tmaps describe the bound E, B, J (3-d, default 4x4x4 block, x extent a multiple of 4)
  int used_tma;    // the last psc_push_particles staged its tiles by TMA tensor copies (psc_store_info)
  Prof prof;
  float q[PSC_MAX_SPECIES], m[PSC_MAX_SPECIES];
  float *E, *B, *J;
  int maxcnt_known;  // PSC_DW_MAXCNT as last read back (psc_refresh_image_size)
  float *rho;      // owned: node charge density of psc_marder ([ext2][ext1][ext0]), lazily allocated
  Cols cols[2];
  int cur;
  int64_t np;
  int32_t np32;    // np as the device sees it (source of an async copy)
  int64_t capacity;  // slots per column the caller bound
  int have_particles, have_fields;
  int state;
  int form;        // PSC_FORM_ABS: absolute positions; PSC_FORM_REL: in-cell offsets
  int xcur;        // exchange[xcur] holds the leavers of the last push (read by the next one)
  int in_step;     // psc_step is calling psc_push_particles (the re-layout check already ran)
  int have_sort_result;  // 1: key/perm/offs_dense describe the last psc_particles_sort
  int bufC;        // StoreDesc::C for the current layout
  // workspace carve-up (all device pointers)
  void *ws;
  size_t ws_bytes;
  int64_t ws_cap;  // max particles the bound workspace was sized for
  int32_t *key, *perm, *cell_idx, *offs_dense, *base, *cnt, *cursor, *big_list, *tot, *doffs, *bigflag;
  uint8_t *bigcell;
  long long *pack, *packloc, *scan_tmp;
  Exchange xch[2];
  Spill spill;
  uint32_t *d_flags;  // owned: PSC_DW_COUNT words
  int64_t launches;
  int last_err;
  int sm_count;
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
static inline bool psc_is3d(const GridDesc &gd) { return gd.n[0] > 1; }

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
int64_t psc_store_capacity(const psc_ctx *c, int64_t n);
int psc_sort_carve(psc_ctx *c, int64_t n);
int psc_sort_general(psc_ctx *c, cudaStream_t s);      // any state -> STORE (stable)
int psc_store_relayout_if_spilled(psc_ctx *c, cudaStream_t s);
int psc_sort_cell_idx(psc_ctx *c, cudaStream_t s);
// dense copy of the store (residents of every cell, then the records waiting in its exchange
// row, then the spill list) into `dst`, keys into `key` (may be null); to_abs: positions absolute
int psc_store_gather(psc_ctx *c, const Cols &dst, int32_t *key, bool to_abs, cudaStream_t s);
StoreDesc psc_store_desc(const psc_ctx *c);
void psc_refresh_image_size(psc_ctx *c, const uint32_t *dw);  // dw: host copy of the status block
// push1.cu / push2.cu
int psc_push_order1(psc_ctx *c, cudaStream_t s);
int psc_make_tile_maps(psc_ctx *c);  // after psc_bind_fields; sets have_tmaps (0 if TMA maps are not applicable)
int psc_push_order2(psc_ctx *c, cudaStream_t s);
// marder.cu
int psc_marder_pass(psc_ctx *c, float diffusion, int iters, cudaStream_t s);
int psc_charge_density_internal(psc_ctx *c, cudaStream_t s);
// balance.cu
int psc_patch_loads_internal(psc_ctx *c, cudaStream_t s, const int32_t patch_blocks[3], int64_t *loads,
                             int32_t np_out[3]);
