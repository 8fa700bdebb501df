// push2.cu -- the fused particle loop of Fig. 8 for second-order
// particles: gather E,B with b2 (TSC) weights (Eq. 11, 31), Boris push
// (Eq. 27-28), move (Eq. 26), Esirkepov charge-conserving deposit, periodic wrap.
//
// One thread block per sort block ("supercell"); a warp takes one CELL at a time
// and walks that cell's particles in chunks of 32, so the cell -- and with it every tile
// address that does not depend on the in-cell offset -- is warp-uniform.  Particle I/O is the
// cell store's (store.cuh): bulk asynchronous copies of the cell's columns into shared memory,
// in-place update, leavers through the exchange rows.
//
// Stencils, relative to the particle's cell l and its in-cell offset a in [0,1) (A13,
// A15).  Because dt <= dx/2 a particle moves less than half a cell, so the node nearest to the
// old AND to the new position is l or l+1, and all b2 weights of both positions live on the four
// nodes l-1 .. l+2:
//   S0[k] = b2(a - k), S1[k] = b2(a + d - k), k = -1..2, DS = S1 - S0   (d = displacement, cells)
// Esirkepov's density decomposition on those nodes, for component c with transverse e, f:
//   W_c[i][je][jf] = DS_c[i] (S0_e S0_f + DS_e S0_f / 2 + S0_e DS_f / 2 + DS_e DS_f / 3)
//                  = DS_c[i] ((S0_e + DS_e/2)(S0_f + DS_f/2) + DS_e DS_f / 12)
//   j_c(i+1/2, je, jf) = j_c(i-1/2, je, jf) - (qw/dV)(dx_c/dt) W_c[i][je][jf],  i = -1, 0, 1
// (the running sum starts from 0 below the stencil and returns to 0 above it because
// sum_i DS[i] = 0).  Along the invariant direction of a 2-d run the current is
// (qw/dV) v_x * bracket.  That is 3 x 48 (3-d) or 16 + 12 + 12 (2-d) current values per
// particle at FIXED offsets from the cell: the 32 lanes' values are summed with a butterfly
// "transpose-reduce" (each stage halves the number of live values per lane) and every lane adds
// its one or two totals to the shared-memory J tile -- no same-address atomic conflicts.
#include <limits.h>

#include "store.cuh"

namespace {

constexpr int PUSH2_THREADS = 256;

// b2 weights of the three points nearest to a sample at distance h in [-1/2, 1/2) from the
// middle point (Eq. 31): points -1, 0, +1.
__device__ __forceinline__ void tsc3(float h, float &wm, float &w0, float &wp) {
  const float a = 0.5f - h, b = 0.5f + h;
  wm = 0.5f * a * a;
  w0 = 0.75f - h * h;
  wp = 0.5f * b * b;
}

// b2 weights of offset a in (-1/2, 3/2) on the nodes -1, 0, 1, 2 relative to the cell
__device__ __forceinline__ void tsc4(float a, float (&S)[4]) {
  const bool up = a >= 0.5f;
  float wm, w0, wp;
  tsc3(up ? a - 1.0f : a, wm, w0, wp);
  S[0] = up ? 0.f : wm;
  S[1] = up ? wm : w0;
  S[2] = up ? w0 : wp;
  S[3] = up ? wp : 0.f;
}

__device__ __forceinline__ float xadd2(bool up, float lo, float hi, int m) {
  return (up ? hi : lo) + __shfl_xor_sync(0xffffffffu, up ? lo : hi, m);
}

// Butterfly transpose-reduce of N per-lane values over the warp.  After the five stages lane L
// holds, in r[0..R), the warp totals of the values with index red_index<N>(L, j) (or padding).
template <int N>
struct RedShape {
  static constexpr int H1 = (N + 1) / 2, H2 = (H1 + 1) / 2, H3 = (H2 + 1) / 2, H4 = (H3 + 1) / 2,
                       H5 = (H4 + 1) / 2;
  static constexpr int R = H5;  // values per lane at the end
};

template <int N, int H>
__device__ __forceinline__ void red_stage(const float (&in)[N], float (&out)[H], bool up, int m) {
#pragma unroll
  for (int i = 0; i < H; i++) out[i] = xadd2(up, in[i], (i + H < N) ? in[i + H] : 0.f, m);
}

template <int N>
__device__ __forceinline__ void warp_reduce_n(const float (&v)[N], float (&r)[RedShape<N>::R],
                                              int lane) {
  using S = RedShape<N>;
  float a[S::H1], b[S::H2], c[S::H3], d[S::H4];
  red_stage<N, S::H1>(v, a, lane & 16, 16);
  red_stage<S::H1, S::H2>(a, b, lane & 8, 8);
  red_stage<S::H2, S::H3>(b, c, lane & 4, 4);
  red_stage<S::H3, S::H4>(c, d, lane & 2, 2);
  red_stage<S::H4, S::H5>(d, r, lane & 1, 1);
}

// The same reduction for the 48 values v[(jf * 4 + je) * 3 + i] of a 3-d current component when
// the caller has filled them from transverse factors ALREADY PERMUTED per lane (perm4 below): a
// lane whose bit 4 (3) is set has its jf index flipped by 2 (1), bit 2 (1) its je index by 2 (1),
// so that in every one of the first four stages each lane keeps the lower half of its values and
// hands the upper half to its partner -- no selects (2 per value and stage otherwise).  The
// totals a lane ends up with are those of warp_reduce_n<48> on the unpermuted values.
__device__ __forceinline__ void warp_reduce_48_permuted(const float (&v)[48], float (&r)[2], int lane) {
  float a[24], b[12], c[6], d[3];
#pragma unroll
  for (int i = 0; i < 24; i++) a[i] = v[i] + __shfl_xor_sync(0xffffffffu, v[i + 24], 16);
#pragma unroll
  for (int i = 0; i < 12; i++) b[i] = a[i] + __shfl_xor_sync(0xffffffffu, a[i + 12], 8);
#pragma unroll
  for (int i = 0; i < 6; i++) c[i] = b[i] + __shfl_xor_sync(0xffffffffu, b[i + 6], 4);
#pragma unroll
  for (int i = 0; i < 3; i++) d[i] = c[i] + __shfl_xor_sync(0xffffffffu, c[i + 3], 2);
  red_stage<3, 2>(d, r, lane & 1, 1);
}

// o[j] = a[j ^ (2 hi + lo)]
__device__ __forceinline__ void perm4(float (&o)[4], const float (&a)[4], bool hi, bool lo) {
  const float t0 = hi ? a[2] : a[0], t1 = hi ? a[3] : a[1], t2 = hi ? a[0] : a[2], t3 = hi ? a[1] : a[3];
  o[0] = lo ? t1 : t0;
  o[1] = lo ? t0 : t1;
  o[2] = lo ? t3 : t2;
  o[3] = lo ? t2 : t3;
}

// index (0..N-1) of the value whose total lane `lane` holds in r[j], or -1 for padding
template <int N>
__device__ __forceinline__ int red_index(int lane, int j) {
  using S = RedShape<N>;
  const int cnt[5] = {N, S::H1, S::H2, S::H3, S::H4};
  const int half[5] = {S::H1, S::H2, S::H3, S::H4, S::H5};
  const int bit[5] = {16, 8, 4, 2, 1};
  int idx = j;  // index inside the last level
  bool ok = true;
#pragma unroll
  for (int l = 4; l >= 0; l--) {
    if (lane & bit[l]) idx += half[l];
    ok = ok && idx < cnt[l];
  }
  return ok ? idx : -1;
}

// CBS != 0: the sort block is CBS cells along every active direction (the library defaults, 8x8
// in 2-d and 4x4x4 in 3-d), so every tile extent and stride folds into an immediate; CBS == 0:
// run-time block.
template <bool D3, int CBS>
struct Geom2 {
  int o[3];     // first cell of the tile
  int bs[3], cpb;
  int te[3];    // tile extents (fields and J alike): bs + 3 points, local point t <-> node o + t - 1
  int tvol;
  __device__ __forceinline__ void init(const GridDesc &gd, int tile) {
    bs[0] = CBS ? (D3 ? CBS : 1) : gd.bs[0];
    bs[1] = CBS ? CBS : gd.bs[1];
    bs[2] = CBS ? CBS : gd.bs[2];
    cpb = bs[0] * bs[1] * bs[2];
    const int b0 = tile % gd.nb[0];
    const int r = tile / gd.nb[0];
    const int b1 = r % gd.nb[1], b2 = r / gd.nb[1];
    o[0] = b0 * bs[0];
    o[1] = b1 * bs[1];
    o[2] = b2 * bs[2];
    te[0] = D3 ? bs[0] + 3 : 1;
    te[1] = bs[1] + 3;
    te[2] = bs[2] + 3;
    tvol = te[0] * te[1] * te[2];
  }
};

// 1-d gather stencils of one particle along one direction
struct Sten2 {
  int tn;           // first tile point of the node-centred stencil (l + (a >= 1/2))
  float wn[3];      // node-centred weights
  float ws[3];      // half-staggered weights; first tile point is l
  // ALT: alternating-order scheme (A29): b1 instead of b2 along a
  // half-staggered direction, on the same three points
  template <bool ALT>
  __device__ __forceinline__ void set(int l, float a) {
    const bool up = a >= 0.5f;
    tn = l + (up ? 1 : 0);
    tsc3(up ? a - 1.0f : a, wn[0], wn[1], wn[2]);
    if (ALT) {
      ws[0] = up ? 0.f : 0.5f - a;
      ws[1] = up ? 1.5f - a : 0.5f + a;
      ws[2] = up ? a - 0.5f : 0.f;
    } else {
      tsc3(a - 0.5f, ws[0], ws[1], ws[2]);
    }
  }
};

template <bool D3, bool SX, bool SY, bool SZ, class TG>
__device__ __forceinline__ float gather2(const float *__restrict__ F, const TG &tg, int lx,
                                         int ly, int lz, const Sten2 &sx, const Sten2 &sy,
                                         const Sten2 &sz) {
  const int ty = SY ? ly : sy.tn, tz = SZ ? lz : sz.tn;
  const float *wy = SY ? sy.ws : sy.wn, *wz = SZ ? sz.ws : sz.wn;
  float acc = 0.f;
  if (D3) {
    const int tx = SX ? lx : sx.tn;
    const float *wx = SX ? sx.ws : sx.wn;
    const float *q = F + (tz * tg.te[1] + ty) * tg.te[0] + tx;
    const int s1 = tg.te[0], s2 = tg.te[0] * tg.te[1];
#pragma unroll
    for (int kz = 0; kz < 3; kz++) {
      float az = 0.f;
#pragma unroll
      for (int ky = 0; ky < 3; ky++) {
        const float *row = q + kz * s2 + ky * s1;
        const float ay = wx[0] * row[0] + wx[1] * row[1] + wx[2] * row[2];
        az = fmaf(wy[ky], ay, az);
      }
      acc = fmaf(wz[kz], az, acc);
    }
  } else {
    const float *q = F + tz * tg.te[1] + ty;
    const int s2 = tg.te[1];
#pragma unroll
    for (int kz = 0; kz < 3; kz++) {
      const float *row = q + kz * s2;
      const float ay = wy[0] * row[0] + wy[1] * row[1] + wy[2] * row[2];
      acc = fmaf(wz[kz], ay, acc);
    }
  }
  return acc;
}

// value layouts of the per-particle current values handed to the reduction
//   3-d, component c (transverse e, f cyclic): v[(jf * 4 + je) * 3 + i]   (48 values)
//   2-d: jx: v[jz * 4 + jy] (16);  jy: v[jz * 3 + i] (12, flux along y);  jz: v[jy * 3 + i] (12)
// tile offset (relative to the cell's own point (lx+1, ly+1, lz+1)) of value `idx`
template <bool D3, class TG>
__device__ __forceinline__ int value_offset(const TG &tg, int comp, int idx) {
  const int s[3] = {1, tg.te[0], tg.te[0] * tg.te[1]};
  if (idx < 0) return INT_MIN;
  if (D3) {
    const int e = (comp + 1) % 3, f = (comp + 2) % 3;
    const int i = idx % 3, je = (idx / 3) % 4, jf = idx / 12;
    return comp * tg.tvol + (i - 1) * s[comp] + (je - 1) * s[e] + (jf - 1) * s[f];
  }
  if (comp == 0) return ((idx / 4) - 1) * s[2] + ((idx % 4) - 1) * s[1];
  if (comp == 1) return tg.tvol + ((idx / 3) - 1) * s[2] + ((idx % 3) - 1) * s[1];
  return 2 * tg.tvol + ((idx % 3) - 1) * s[2] + ((idx / 3) - 1) * s[1];
}

// BIG == false: the cells that fit the shared-memory image (store.cuh); BIG == true: a second
// launch for the tiles in which the first one had to leave a cell out.
template <bool D3, int CBS, bool XC, bool BIG, bool ALT>
__global__ void __launch_bounds__(PUSH2_THREADS, 2)
k_push2(GridDesc gd, StoreDesc sd, const float *__restrict__ E, const float *__restrict__ B,
        float *__restrict__ J, int wstride) {
  extern __shared__ __align__(128) unsigned char smraw[];
  // the image launch has one block per tile; the BIG launch a few blocks that walk the flagged tiles
#pragma unroll 1
  if (BIG) {
    if (blockIdx.x == 0 && threadIdx.x == 0) *sd.nbig_next = 0;
    if (*sd.nbig == 0) return;  // the image launch left nothing out
  }
  for (int tile = blockIdx.x;; tile += gridDim.x) {
  if (BIG) {
    if (tile >= gd.ntiles) break;
    if (!sd.bigflag[tile]) continue;
  }
  using Walker = CellWalker<D3, XC, BIG>;
  Geom2<D3, CBS> tg;
  tg.init(gd, tile);
  const int lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
  // (broadcast from lane 0: lets the compiler keep everything derived from the warp index uniform)
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
  float *sF = (float *)(smraw + (size_t)nwarps * wstride);  // [6][tvol]
  float *sJ = sF + 6 * tg.tvol;                              // [3][tvol]
  float *sH = sJ + 3 * tg.tvol;                              // [8]: Boris h per species
  int *sNbT = (int *)(sH + PSC_MAX_SPECIES);                 // [27]: first key of the 3^3 neighbouring tiles
  int *sBase = sNbT + 27;                                    // [cpb + 1]
  int *sCnt = sBase + tg.cpb + 1;                            // [cpb]
  Walker wk;
  wk.init(smraw + (size_t)warp * wstride, sd, lane, sNbT);
  const int kbase = tile * tg.cpb;
  // the resident run of the warp's first cell is requested before anything else: its DRAM latency
  // passes while the block stages its field tile
  if (!BIG && warp < tg.cpb) wk.issue_loads(sd, sd.cnt[kbase + warp], sd.base[kbase + warp]);
  if (threadIdx.x < 27) {  // periodic neighbour tiles (the single-GPU particle exchange)
    const int t = threadIdx.x;
    const int b0 = tile % gd.nb[0], br = tile / gd.nb[0];
    const int b1 = br % gd.nb[1], b2 = br / gd.nb[1];
    const int n0 = wrap_cell(b0 + t % 3 - 1, gd.nb[0]), n1 = wrap_cell(b1 + (t / 3) % 3 - 1, gd.nb[1]),
              n2 = wrap_cell(b2 + t / 9 - 1, gd.nb[2]);
    sNbT[t] = ((n2 * gd.nb[1] + n1) * gd.nb[0] + (D3 ? n0 : 0)) * tg.cpb;
  }

  if (threadIdx.x < PSC_MAX_SPECIES) sH[threadIdx.x] = gd.qmh[threadIdx.x];
  // (asynchronous copies: all of a thread's requests are in flight together)
  for (int i = threadIdx.x; i <= tg.cpb; i += blockDim.x) {
    cp_async4(sBase + i, sd.base + kbase + i, true);
    if (i < tg.cpb) cp_async4(sCnt + i, sd.cnt + kbase + i, true);
  }
  for (int i = threadIdx.x; i < 6 * tg.tvol; i += blockDim.x) {
    const int c = i / tg.tvol, r = i - c * tg.tvol;
    const int tx = r % tg.te[0], t = r / tg.te[0];
    const int ty = t % tg.te[1], tz = t / tg.te[1];
    const int gx = D3 ? tg.o[0] + tx - 1 + gd.g[0] : 0;
    const int gy = tg.o[1] + ty - 1 + gd.g[1], gz = tg.o[2] + tz - 1 + gd.g[2];
    const int gi = (gz * gd.ext[1] + gy) * gd.ext[0] + gx;
    cp_async4(sF + i, c < 3 ? E + c * gd.comp + gi : B + (c - 3) * gd.comp + gi, true);
  }
  cp_async_commit();
  for (int i = threadIdx.x; i < 3 * tg.tvol; i += blockDim.x) sJ[i] = 0.f;

  // which totals this lane holds after each reduction, as J-tile offsets from the cell's point
  constexpr int NX = D3 ? 48 : 16, NY = D3 ? 48 : 12, NZ = D3 ? 48 : 12;
  int offx[2], offy[2], offz[2];
#pragma unroll
  for (int j = 0; j < 2; j++) {
    offx[j] = j < RedShape<NX>::R ? value_offset<D3>(tg, 0, red_index<NX>(lane, j)) : INT_MIN;
    offy[j] = j < RedShape<NY>::R ? value_offset<D3>(tg, 1, red_index<NY>(lane, j)) : INT_MIN;
    offz[j] = j < RedShape<NZ>::R ? value_offset<D3>(tg, 2, red_index<NZ>(lane, j)) : INT_MIN;
  }
  cp_async_wait<0>();
  __syncthreads();

  const float *sEx = sF, *sEy = sF + tg.tvol, *sEz = sF + 2 * tg.tvol;
  const float *sBx = sF + 3 * tg.tvol, *sBy = sF + 4 * tg.tvol, *sBz = sF + 5 * tg.tvol;
  uint32_t bad = 0;

  // The move x^{n+1/2} -> x^{n+3/2} (Eq. 26) in cells, written with explicit roundings: the pass
  // over a cell's leavers recomputes it from the stored momentum and must get the same bits.
  const float cdx = D3 ? gd.dt_dx[0] : 0.f, cdy = gd.dt_dx[1], cdz = gd.dt_dx[2];
  auto move = [&](float ax, float ay, float az, float ux, float uy, float uz, float &vx, float &endx,
                  float &endy, float &endz) {
    const float ig = rsqrt_ge1(__fmaf_rn(ux, ux, __fmaf_rn(uy, uy, __fmaf_rn(uz, uz, 1.0f))));
    vx = __fmul_rn(ux, ig);
    endx = D3 ? __fmaf_rn(vx, cdx, ax) : ax;
    endy = __fmaf_rn(__fmul_rn(uy, ig), cdy, ay);
    endz = __fmaf_rn(__fmul_rn(uz, ig), cdz, az);
  };
  // a particle that leaves its cell: its record (offsets relative to the destination cell) goes
  // to the cell's exchange row
  auto depart = [&](bool leave, int xi, int lx, int ly, int lz, float ax, float ay, float az, float endx,
                    float endy, float endz, float ux, float uy, float uz, float qw, int sp, float x2d, int id) {
    if (leave) {
      const int sxd = D3 ? (endx >= 1.f ? 1 : (endx < 0.f ? -1 : 0)) : 0;
      const int syd = endy >= 1.f ? 1 : (endy < 0.f ? -1 : 0);
      const int szd = endz >= 1.f ? 1 : (endz < 0.f ? -1 : 0);
      // a non-finite end position (PSC_F_NAN) compares false everywhere: the particle keeps its old
      // offsets and returns to its own cell through the spill list instead of being dropped
      const bool nowhere = (sxd | syd | szd) == 0;
      Part pr;
      pr.ax = D3 ? fminf(fmaxf(endx - (float)sxd, 0.f), 0.99999994f) : 0.f;
      pr.ay = fminf(fmaxf(endy - (float)syd, 0.f), 0.99999994f);
      pr.az = fminf(fmaxf(endz - (float)szd, 0.f), 0.99999994f);
      if (nowhere) { pr.ax = D3 ? ax : 0.f; pr.ay = ay; pr.az = az; }
      pr.ux = ux; pr.uy = uy; pr.uz = uz; pr.qw = qw; pr.sp = sp;
      float w[8];
      Walker::to_words(w, pr, x2d);
      int dest = 0;
      if (xi >= PSC_XCAP || nowhere)
        dest = cell_key(gd, D3 ? wrap_cell(tg.o[0] + lx + sxd, gd.n[0]) : 0,
                        wrap_cell(tg.o[1] + ly + syd, gd.n[1]), wrap_cell(tg.o[2] + lz + szd, gd.n[2]));
      wk.emit(sd, nowhere ? PSC_XCAP : xi, dir_code<D3>(sxd, syd, szd), w, id, dest);
    }
  };

  int src_next;
  unsigned mask_next = wk.fetch_mask(sd, tg, warp, src_next);
#pragma unroll 1
  for (int ci = warp; ci < tg.cpb; ci += nwarps) {
    const int nx = ci + nwarps;
    const int next_n = nx < tg.cpb ? sCnt[nx] : 0, next_base = nx < tg.cpb ? sBase[nx] : 0;
    const unsigned mask = mask_next;
    const int src = src_next;
    mask_next = wk.fetch_mask(sd, tg, nx, src_next);
    wk.begin_cell(kbase + ci, sCnt[ci], sBase[ci], sBase[ci + 1] - sBase[ci], mask, src);
    // Whose cell is it?  The image launch decides (its count is the one before the push) and
    // leaves a note; the BIG launch takes exactly the noted cells.
    if (BIG) {
      if (!sd.bigcell[kbase + ci]) continue;
      __syncwarp();
      if (lane == 0) sd.bigcell[kbase + ci] = 0;
    } else if (!wk.fits) {
      if (lane == 0) {  // note the cell and (once) its tile for the BIG launch
        sd.bigcell[kbase + ci] = 1;
        if (atomicExch(&sd.bigflag[tile], 1) == 0) atomicAdd(sd.nbig, 1u);
      }
      wk.skip_cell(sd, next_n, next_base);
      continue;
    }
    const int lx = ci % tg.bs[0], lt = ci / tg.bs[0];
    const int ly = lt % tg.bs[1], lz = lt / tg.bs[1];
    const int np_cell = wk.n + wk.na;  // residents + arrivals (reorder on load)
    float *cellJ = sJ + (D3 ? ((lz + 1) * tg.te[1] + (ly + 1)) * tg.te[0] + (lx + 1)
                            : (lz + 1) * tg.te[1] + (ly + 1));
    if (!BIG && wk.na) wk.stage_arrivals(sd);
    bool landed = false;
    // the lane's reduced totals, summed over the chunks of the cell: one shared-memory add per
    // cell instead of one per chunk (a shared fp32 atomicAdd is a compare-and-swap loop)
    float racc[3][2] = {{0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}};
#pragma unroll 1
    for (int base = 0; base < np_cell; base += 32) {
      Part cur;
      float x2d = 0.f;
      int id = 0;
      bool act;
      if (BIG) {
        act = wk.load_global(sd, base, cur, x2d, id);
      } else {
        if (!landed && base + 32 > wk.n) {
          wk.arrivals_landed();
          landed = true;
        }
        act = base + lane < np_cell;
        wk.load_image(base + lane, cur);
      }
      const float ax = D3 ? cur.ax : 0.25f, ay = cur.ay, az = cur.az;
      float ux = cur.ux, uy = cur.uy, uz = cur.uz;
      const float qw = act ? cur.qw : 0.f;
      const int sp = cur.sp & (PSC_MAX_SPECIES - 1);
      // ---- gather (Eq. 11 with b2 weights; each component from its own Yee points) ---------
      Sten2 sx, sy, sz;
      sx.template set<ALT>(lx, ax);
      sy.template set<ALT>(ly, ay);
      sz.template set<ALT>(lz, az);
      const float ex = gather2<D3, true, false, false>(sEx, tg, lx, ly, lz, sx, sy, sz);
      const float ey = gather2<D3, false, true, false>(sEy, tg, lx, ly, lz, sx, sy, sz);
      const float ez = gather2<D3, false, false, true>(sEz, tg, lx, ly, lz, sx, sy, sz);
      const float bx = gather2<D3, false, true, true>(sBx, tg, lx, ly, lz, sx, sy, sz);
      const float by = gather2<D3, true, false, true>(sBy, tg, lx, ly, lz, sx, sy, sz);
      const float bz = gather2<D3, true, true, false>(sBz, tg, lx, ly, lz, sx, sy, sz);

      // ---- Boris (Eq. 27-28) and move (Eq. 26) ----------------------------------------------
      boris_push(ux, uy, uz, ex, ey, ez, bx, by, bz, sH[sp]);
      float vx, endx, endy, endz;
      move(ax, ay, az, ux, uy, uz, vx, endx, endy, endz);

      // ---- Esirkepov deposit ------------------------------------------------------------------
      {
        float S0[4], S1[4];
        float Ym[4], Yd[4], Zm[4], Zd[4];  // S0 + DS/2 and DS along y, z
        float Ay[3], Az[3];                // running sums -f * DS along y, z
        tsc4(ay, S0);
        tsc4(endy, S1);
        {
          const float f = qw * gd.cur[1];
          float run = 0.f;
#pragma unroll
          for (int k = 0; k < 4; k++) {
            Yd[k] = S1[k] - S0[k];
            Ym[k] = S0[k] + 0.5f * Yd[k];
            if (k < 3) { run -= f * Yd[k]; Ay[k] = run; }
          }
        }
        tsc4(az, S0);
        tsc4(endz, S1);
        {
          const float f = qw * gd.cur[2];
          float run = 0.f;
#pragma unroll
          for (int k = 0; k < 4; k++) {
            Zd[k] = S1[k] - S0[k];
            Zm[k] = S0[k] + 0.5f * Zd[k];
            if (k < 3) { run -= f * Zd[k]; Az[k] = run; }
          }
        }
        if (D3) {
          float Xm[4], Xd[4], Ax[3];
          tsc4(ax, S0);
          tsc4(endx, S1);
          {
            const float f = qw * gd.cur[0];
            float run = 0.f;
#pragma unroll
            for (int k = 0; k < 4; k++) {
              Xd[k] = S1[k] - S0[k];
              Xm[k] = S0[k] + 0.5f * Xd[k];
              if (k < 3) { run -= f * Xd[k]; Ax[k] = run; }
            }
          }
          // one component at a time: 48 values A_c[i] * (Em[je] Fm[jf] + Ed[je] Fd[jf] / 12) from the
          // transverse factors permuted for the select-free reduction (e-role: lane bits 2, 1;
          // f-role: lane bits 4, 3)
          const bool l4 = lane & 16, l3 = lane & 8, l2 = lane & 4, l1 = lane & 2;
          auto component = [&](const float (&A)[3], const float (&Em)[4], const float (&Ed)[4],
                               const float (&Fm)[4], const float (&Fd)[4], float (&rsum)[2]) {
            float em[4], ed[4], fm[4], fd[4];
            perm4(em, Em, l2, l1);
            perm4(ed, Ed, l2, l1);
            perm4(fm, Fm, l4, l3);
            perm4(fd, Fd, l4, l3);
#pragma unroll
            for (int k = 0; k < 4; k++) fd[k] *= (1.0f / 12.0f);
            float v[48];
#pragma unroll
            for (int jf = 0; jf < 4; jf++)
#pragma unroll
              for (int je = 0; je < 4; je++) {
                const float br = fmaf(em[je], fm[jf], ed[je] * fd[jf]);
#pragma unroll
                for (int i = 0; i < 3; i++) v[(jf * 4 + je) * 3 + i] = A[i] * br;
              }
            float r[2];
            warp_reduce_48_permuted(v, r, lane);
            rsum[0] += r[0];
            rsum[1] += r[1];
          };
          component(Ax, Ym, Yd, Zm, Zd, racc[0]);  // jx: transverse e = y, f = z
          component(Ay, Zm, Zd, Xm, Xd, racc[1]);  // jy: e = z, f = x
          component(Az, Xm, Xd, Ym, Yd, racc[2]);  // jz: e = x, f = y
        } else {
          const float qvx = qw * gd.inv_dV * vx;
          {
            float v[16];
#pragma unroll
            for (int jz = 0; jz < 4; jz++)
#pragma unroll
              for (int jy = 0; jy < 4; jy++)
                v[jz * 4 + jy] = qvx * fmaf(Ym[jy], Zm[jz], Yd[jy] * Zd[jz] * (1.0f / 12.0f));
            float r[RedShape<16>::R];
            warp_reduce_n<16>(v, r, lane);
#pragma unroll
            for (int j = 0; j < RedShape<16>::R; j++) racc[0][j] += r[j];
          }
          {
            float v[12];
#pragma unroll
            for (int jz = 0; jz < 4; jz++)
#pragma unroll
              for (int i = 0; i < 3; i++) v[jz * 3 + i] = Ay[i] * Zm[jz];
            float r[RedShape<12>::R];
            warp_reduce_n<12>(v, r, lane);
#pragma unroll
            for (int j = 0; j < RedShape<12>::R; j++) racc[1][j] += r[j];
          }
          {
            float v[12];
#pragma unroll
            for (int jy = 0; jy < 4; jy++)
#pragma unroll
              for (int i = 0; i < 3; i++) v[jy * 3 + i] = Az[i] * Ym[jy];
            float r[RedShape<12>::R];
            warp_reduce_n<12>(v, r, lane);
#pragma unroll
            for (int j = 0; j < RedShape<12>::R; j++) racc[2][j] += r[j];
          }
        }
      }

      // ---- file the particle: in place if it stays; a leaver is noted (image path) or recorded
      const bool stay = (!D3 || (endx >= 0.f && endx < 1.f)) && endy >= 0.f && endy < 1.f &&
                        endz >= 0.f && endz < 1.f;
      const bool leave = act && !stay;
      Part pn;
      pn.ax = endx; pn.ay = endy; pn.az = endz;
      pn.ux = ux; pn.uy = uy; pn.uz = uz; pn.qw = qw; pn.sp = sp;
      if (BIG) {
        if (__any_sync(0xffffffffu, leave)) {
          const int xi = wk.leaver_slot(leave);
          depart(leave, xi, lx, ly, lz, ax, ay, az, endx, endy, endz, ux, uy, uz, qw, sp, x2d, id);
        }
        wk.store_global(sd, act && stay, pn, x2d, id);
      } else {
        wk.store_image(base, act, leave, pn);
      }
      if (act && !(fabsf(ux) + fabsf(uy) + fabsf(uz) < 3.0e38f)) bad |= PSC_F_NAN;
    }
#pragma unroll
    for (int j = 0; j < 2; j++) {
      if (offx[j] != INT_MIN) atomicAdd(cellJ + offx[j], racc[0][j]);
      if (offy[j] != INT_MIN) atomicAdd(cellJ + offy[j], racc[1][j]);
      if (offz[j] != INT_MIN) atomicAdd(cellJ + offz[j], racc[2][j]);
    }
    if (BIG) {
      wk.end_global(sd);
    } else {
      // the records of the cell's leavers, 32 at a time (their deposit is done: Esirkepov's
      // stencil covers the move across the face)
      const int nl = wk.nh;
#pragma unroll 1
      for (int i0 = 0; i0 < nl; i0 += 32) {
        const bool al = i0 + lane < nl;
        Part q;
        float qx2d = 0.f;
        int qid = 0;
        q.ax = q.ay = q.az = 0.25f; q.ux = q.uy = q.uz = q.qw = 0.f; q.sp = 0;
        if (al) wk.leaver(sd, i0 + lane, q, qx2d, qid);
        float qvx, qex, qey, qez;
        move(D3 ? q.ax : 0.25f, q.ay, q.az, q.ux, q.uy, q.uz, qvx, qex, qey, qez);
        depart(al, i0 + lane, lx, ly, lz, q.ax, q.ay, q.az, qex, qey, qez, q.ux, q.uy, q.uz, q.qw,
               q.sp & (PSC_MAX_SPECIES - 1), qx2d, qid);
      }
      wk.end_image(sd, next_n, next_base);
    }
  }
  wk.finish();
  if (bad) atomicOr(sd.flags, bad);
  __syncthreads();
  if (BIG && threadIdx.x == 0) sd.bigflag[tile] = 0;  // taken care of: the flag is the image launch's to set

  // ---- flush the J tile to global J -----------------------------------------------------------
  for (int i = threadIdx.x; i < 3 * tg.tvol; i += blockDim.x) {
    const float v = sJ[i];
    if (v == 0.f) continue;
    const int c = i / tg.tvol, r = i - c * tg.tvol;
    const int tx = r % tg.te[0], t = r / tg.te[0];
    const int ty = t % tg.te[1], tz = t / tg.te[1];
    const int gx = D3 ? tg.o[0] + tx - 1 + gd.g[0] : 0;
    const int gy = tg.o[1] + ty - 1 + gd.g[1], gz = tg.o[2] + tz - 1 + gd.g[2];
    atomicAdd(&J[c * gd.comp + (gz * gd.ext[1] + gy) * gd.ext[0] + gx], v);
  }
  if (!BIG) break;
  __syncthreads();  // the next tile reuses the shared memory
  }
}

}  // namespace

int psc_push_order2(psc_ctx *c, cudaStream_t s) {
  const GridDesc &gd = c->gd;
  const bool d3 = gd.n[0] > 1 && gd.n[1] > 1 && gd.n[2] > 1;
  const bool d2yz = gd.n[0] == 1 && gd.n[1] > 1 && gd.n[2] > 1;
  if (!d3 && !d2yz) return PSC_ERR_UNSUPPORTED;  // 2-d runs are yz-plane runs (A25)
  int tvol = 1;
  for (int d = 0; d < 3; d++)
    if (gd.n[d] > 1) tvol *= gd.bs[d] + 3;
  const StoreDesc sd = psc_store_desc(c);
  const bool xc = sd.icol_id >= 0 || sd.icol_x2d >= 0;
  const int threads = PUSH2_THREADS;
  auto stride = [&](int wbytes) { return (wbytes + 127) / 128 * 128; };
  const int ws_img = stride(d3 ? CellWalker<true, true, false>::smem_bytes(sd.imgC, sd.ncol)
                               : CellWalker<false, true, false>::smem_bytes(sd.imgC, sd.ncol));
  const int ws_big = stride(CellWalker<true, true, true>::smem_bytes(sd.imgC, sd.ncol));
  const size_t tile_bytes = (size_t)(9 * tvol + PSC_MAX_SPECIES + 27 + 2 * gd.cpb + 2) * sizeof(float);
  const size_t smem_img = (size_t)(threads / 32) * ws_img + tile_bytes;
  const size_t smem_big = (size_t)(threads / 32) * ws_big + tile_bytes;
  if (smem_img > 200 * 1024) return PSC_ERR_UNSUPPORTED;
  const int big_grid = gd.ntiles < 2 * c->sm_count ? gd.ntiles : 2 * c->sm_count;
  ProfScope ps(c, PSC_PH_PUSH, s);
#define PSC_LAUNCH_PUSH2_(D3_, CBS_, XC_, BIG_, SMEM_, WS_)                                         \
  do {                                                                                             \
    PSC_CUDA_TRY(c, cudaFuncSetAttribute(k_push2<D3_, CBS_, XC_, BIG_, false>,                     \
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(SMEM_))); \
    k_push2<D3_, CBS_, XC_, BIG_, false><<<(BIG_) ? big_grid : gd.ntiles, threads, SMEM_, s>>>(gd, sd, c->E, c->B, c->J, WS_); \
    PSC_LAUNCH_CHECK(c);                                                                           \
  } while (0)
  // the alternating-order scheme runs the general instantiation (run-time tile, optional columns)
#define PSC_LAUNCH_PUSH2_ALT(D3_, BIG_, SMEM_, WS_)                                                 \
  do {                                                                                             \
    PSC_CUDA_TRY(c, cudaFuncSetAttribute(k_push2<D3_, 0, true, BIG_, true>,                        \
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(SMEM_))); \
    k_push2<D3_, 0, true, BIG_, true><<<(BIG_) ? big_grid : gd.ntiles, threads, SMEM_, s>>>(gd, sd, c->E, c->B, c->J, WS_); \
    PSC_LAUNCH_CHECK(c);                                                                           \
  } while (0)
#define PSC_LAUNCH_PUSH2(D3_, CBS_)                                       \
  do {                                                                    \
    if (xc) {                                                             \
      PSC_LAUNCH_PUSH2_(D3_, CBS_, true, false, smem_img, ws_img);        \
      PSC_LAUNCH_PUSH2_(D3_, CBS_, true, true, smem_big, ws_big);         \
    } else {                                                              \
      PSC_LAUNCH_PUSH2_(D3_, CBS_, false, false, smem_img, ws_img);       \
      PSC_LAUNCH_PUSH2_(D3_, CBS_, false, true, smem_big, ws_big);        \
    }                                                                     \
  } while (0)
  if (gd.gmode == PSC_SCHEME_ALTERNATING) {
    if (d3) {
      PSC_LAUNCH_PUSH2_ALT(true, false, smem_img, ws_img);
      PSC_LAUNCH_PUSH2_ALT(true, true, smem_big, ws_big);
    } else {
      PSC_LAUNCH_PUSH2_ALT(false, false, smem_img, ws_img);
      PSC_LAUNCH_PUSH2_ALT(false, true, smem_big, ws_big);
    }
  } else if (d3) {
    if (gd.bs[0] == 4 && gd.bs[1] == 4 && gd.bs[2] == 4) PSC_LAUNCH_PUSH2(true, 4);
    else PSC_LAUNCH_PUSH2(true, 0);
  } else {
    if (gd.bs[1] == 8 && gd.bs[2] == 8) PSC_LAUNCH_PUSH2(false, 8);
    else PSC_LAUNCH_PUSH2(false, 0);
  }
#undef PSC_LAUNCH_PUSH2
#undef PSC_LAUNCH_PUSH2_
#undef PSC_LAUNCH_PUSH2_ALT
  return PSC_OK;
}
