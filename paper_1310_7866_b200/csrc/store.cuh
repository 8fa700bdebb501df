// store.cuh -- device side of the cell store (psc_internal.cuh): how a warp
// streams one cell's particles through shared memory.
//
// a particle moves at most one cell per step, so the per-step "sort" only has to
// deal with the few particles that change cell, and the reorder can be folded into the next
// push's load ("only one loop each time step that reads and writes all particle data").  Here:
//   * a cell's resident particles are one 128-byte-aligned run per column; the warp that owns the
//     cell fetches the whole run with ONE bulk asynchronous copy per column (cp.async.bulk ->
//     UBLKCP: issued by one lane, executed by the copy engine, completion counted on an mbarrier),
//     so the SM's load/store pipe never sees the particle stream;
//   * the warp advances the particles in that shared-memory image IN PLACE, and writes the image's
//     dynamic columns (positions, momenta) back with one bulk copy per column; q*w, species, id of
//     a particle that stays in its cell are never rewritten.  A resident that leaves keeps its OLD
//     offsets in the image next to its NEW momentum and is only noted in the hole list; once all
//     residents of the cell are done, one pass over that list (32 leavers at a time instead of one
//     or two per chunk) recomputes the move bit-identically, writes the records and deposits;
//   * a particle that leaves is appended, as one 32-byte record, to the exchange row of its
//     SOURCE cell (ping-pong buffered); the row's header holds one 32-bit mask per direction code
//     (9 / 27 destination classes) saying which records moved that way;
//   * the arrivals of a cell are the records of its 8 / 26 neighbours' rows whose direction points
//     at it: one 4-byte header load per neighbour finds them (requested one cell ahead), and
//     asynchronous 4-byte copies (cp.async) drop their words into the image BEHIND the residents
//     while the residents are being pushed -- from then on an arrival is a particle of the cell
//     like any other (reorder on load);
//   * at the end of the cell the holes the leavers left are closed by moving particles from the
//     tail of the image, so that [0, cnt) stays dense.
// A cell that does not fit the image (more than C particles incl. arrivals) is left to a second
// launch of the same kernel in its BIG form, which streams such cells straight from and to global
// memory with an in-place compaction (rare; correct for any size; tiles without such a cell leave
// at once).  A particle that finds no room (row or cell full) goes to the spill list; the next
// step files it into its cell if that has room by then, else re-lays the store out (sort.cu).
#pragma once
#include "push_common.cuh"

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *b, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *b, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *b, unsigned parity) {
  unsigned ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok)
      : "r"(smem_u32(b)), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t *b, unsigned parity) {
  while (!mbar_try_wait(b, parity)) {
  }
}
// global -> shared bulk copy (16-byte aligned, size a multiple of 16), completion on `bar`
__device__ __forceinline__ void bulk_g2s(void *sdst, const void *gsrc, unsigned bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(sdst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// shared -> global bulk copy, tracked by the issuing thread's bulk group
__device__ __forceinline__ void bulk_s2g(void *gdst, const void *ssrc, unsigned bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
               ::"l"(gdst), "r"(smem_u32(ssrc)), "r"(bytes) : "memory");
}
// TMA tensor copies (4-d tiled tensor map): global box at coordinates (c0, c1, c2, c3) -> shared
// (128-byte aligned), completion on `bar`; shared -> global with element-wise add
__device__ __forceinline__ void tma_load_4d(void *sdst, const void *map, int c0, int c1, int c2, int c3,
                                            uint64_t *bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
      ::"r"(smem_u32(sdst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_reduce_add_4d(const void *map, const void *ssrc, int c0, int c1, int c2,
                                                  int c3) {
  asm volatile("cp.reduce.async.bulk.tensor.4d.global.shared::cta.add.tile.bulk_group [%0, {%2, %3, %4, %5}], [%1];"
               ::"l"(map), "r"(smem_u32(ssrc)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// cell key (block-major, cell-minor) of periodic cell coordinates
__device__ __forceinline__ int wrap_cell(int c, int n) { return c < 0 ? c + n : (c >= n ? c - n : c); }
__device__ __forceinline__ int cell_key(const GridDesc &gd, int cx, int cy, int cz) {
  if ((gd.bsh[0] | gd.bsh[1] | gd.bsh[2]) >= 0) {  // power-of-two blocks (the defaults): shifts
    const int b0 = cx >> gd.bsh[0], b1 = cy >> gd.bsh[1], b2 = cz >> gd.bsh[2];
    const int l0 = cx & (gd.bs[0] - 1), l1 = cy & (gd.bs[1] - 1), l2 = cz & (gd.bs[2] - 1);
    return ((b2 * gd.nb[1] + b1) * gd.nb[0] + b0) * gd.cpb + (((l2 << gd.bsh[1]) + l1) << gd.bsh[0]) + l0;
  }
  const int b0 = cx / gd.bs[0], b1 = cy / gd.bs[1], b2 = cz / gd.bs[2];
  const int l0 = cx - b0 * gd.bs[0], l1 = cy - b1 * gd.bs[1], l2 = cz - b2 * gd.bs[2];
  return ((b2 * gd.nb[1] + b1) * gd.nb[0] + b0) * gd.cpb + (l2 * gd.bs[1] + l1) * gd.bs[0] + l0;
}
// key -> cell coordinates
__device__ __forceinline__ void key_to_cell(const GridDesc &gd, int k, int c[3]) {
  if ((gd.bsh[0] | gd.bsh[1] | gd.bsh[2]) >= 0) {  // power-of-two blocks: shifts for the in-block part
    const int sh01 = gd.bsh[0] + gd.bsh[1];
    const int b = k >> (sh01 + gd.bsh[2]), l = k & (gd.cpb - 1);
    const int b0 = b % gd.nb[0], br = b / gd.nb[0];
    const int b1 = br % gd.nb[1], b2 = br / gd.nb[1];
    c[0] = (b0 << gd.bsh[0]) + (l & (gd.bs[0] - 1));
    c[1] = (b1 << gd.bsh[1]) + ((l >> gd.bsh[0]) & (gd.bs[1] - 1));
    c[2] = (b2 << gd.bsh[2]) + (l >> sh01);
    return;
  }
  const int b = k / gd.cpb, l = k - b * gd.cpb;
  const int b0 = b % gd.nb[0], br = b / gd.nb[0];
  const int b1 = br % gd.nb[1], b2 = br / gd.nb[1];
  const int l0 = l % gd.bs[0], lr = l / gd.bs[0];
  const int l1 = lr % gd.bs[1], l2 = lr / gd.bs[1];
  c[0] = b0 * gd.bs[0] + l0;
  c[1] = b1 * gd.bs[1] + l1;
  c[2] = b2 * gd.bs[2] + l2;
}

template <bool D3>
__device__ __forceinline__ void dir_decode(int dc, int &sx, int &sy, int &sz) {
  if (D3) {
    sx = dc % 3 - 1;
    sy = (dc / 3) % 3 - 1;
    sz = dc / 9 - 1;
  } else {
    sx = 0;
    sy = dc % 3 - 1;
    sz = dc / 3 - 1;
  }
}

// a particle that found no room in its exchange row or its destination cell
static __device__ __noinline__ void spill_record(Spill sp, uint32_t *flags, int key, uint4 a, uint4 b, int id) {
  const int i = atomicAdd(sp.count, 1);
  if (i < sp.cap) {
    XRec r;
    r.a = a;
    r.b = b;
    sp.rec[i] = r;
    sp.key[i] = key;
    if (sp.id) sp.id[i] = id;
  } else {
    atomicOr(flags, PSC_F_OVERFLOW);  // the particle is lost: the workspace was sized for fewer particles
  }
}
__device__ __forceinline__ void spill_particle(const StoreDesc &sd, int key, const float (&w)[8], int id) {
  spill_record(sd.spill, sd.flags, key,
               make_uint4(__float_as_uint(w[0]), __float_as_uint(w[1]), __float_as_uint(w[2]), __float_as_uint(w[3])),
               make_uint4(__float_as_uint(w[4]), __float_as_uint(w[5]), __float_as_uint(w[6]), __float_as_uint(w[7])), id);
}

// One particle in registers: in-cell offsets a*, momenta, the static values.
struct Part {
  float ax, ay, az, ux, uy, uz, qw;
  int sp;
};

constexpr int WALK_AC = 128;  // arrival-list window (entries)
constexpr int WALK_HC = 128;  // hole-list entries kept as bytes (more holes are read off the bitmap)

// Per-warp view of the store.  XC: optional columns (id, carried x of a 2-d run) may be bound.
// BIG == false: the shared-memory image path (cells with n + arrivals <= C; others are skipped
// and reported); BIG == true: the global-memory path for exactly those others.
// CT != 0: the image has CT slots per column (a compile-time stride folds the column offsets of
// every image access into immediates); CT == 0: the stride is the run-time sd.imgC.
template <bool D3, bool XC, bool BIG, int CT = 0>
struct CellWalker {
  static constexpr int ND = D3 ? 27 : 9, STAY = D3 ? 13 : 4, NDYN = D3 ? 6 : 5, NREC = D3 ? 8 : 7;
  static constexpr int XW = D3 ? PSC_XW3 : PSC_XW2;  // header words of an exchange row
  // bytes of per-warp shared memory for an image of C slots x ncol columns
  __host__ __device__ static constexpr int smem_bytes(int C, int ncol) {
    return (BIG ? WALK_AC * 2 /*arr*/ + 32 * 4 /*nbk*/ : ncol * C * 4 + WALK_HC /*holes*/) + XW * 4 /*xrow*/ +
           12 * 4 /*hbm*/ + 16 /*bar*/;
  }
  float *buf;      // [ncol][C]
  uint8_t *holes;  // [WALK_HC]: slots of the image whose particle left, ascending (the first WALK_HC)
  uint16_t *arr;   // [WALK_AC]: arrival a -> direction lane << 8 | record index in that neighbour's row
  int *nbk;        // [32]: key of the neighbour cell a lane looks at
  unsigned *xrow;  // [XW]: per direction code, which of the cell's records so far moved that way
  unsigned *hbm;   // [12] (9 used): bit v set <=> slot v of the image is a hole; hbm[11]: arrival counter
  int *acnt;
  uint64_t *bar;
  const int *nbt;  // [27] (block-wide): first key of the tile at tile offset (tx, ty, tz) in {-1,0,1}^3
  int Crt, ncol, lane;
#define C (CT ? CT : Crt)
  unsigned lt;
  unsigned parity;
  bool loads_armed;  // bulk loads for the cell about to be processed are in flight
  // current cell
  int key, n, na, base, cap;
  bool fits;         // n + na <= C: the cell takes the image path
  int nh, tcur, nleave, a0, my_start, my_src;
  unsigned my_mask;

  __device__ __forceinline__ void init(unsigned char *wsm, const StoreDesc &sd, int lane_, const int *nbt_) {
    Crt = sd.imgC;
    ncol = XC ? sd.ncol : NREC;
    lane = lane_;
    nbt = nbt_;
    lt = lanemask_lt_();
    buf = (float *)wsm;
    holes = (uint8_t *)(buf + (BIG ? 0 : ncol * C));
    arr = (uint16_t *)(holes + (BIG ? 0 : WALK_HC));  // (arr, nbk: the BIG form only)
    nbk = (int *)(arr + (BIG ? WALK_AC : 0));
    xrow = (unsigned *)(nbk + (BIG ? 32 : 0));
    hbm = xrow + XW;
    bar = (uint64_t *)(hbm + 12);
    acnt = (int *)(hbm + 11);
    if (lane == 0) *acnt = 0;
    parity = 0;
    loads_armed = false;
    if (lane < XW) xrow[lane] = 0u;
    if (!BIG && lane == 0) {
      mbar_init(bar, 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
  }

  // lane 0: fetch the resident run of a cell into the image (n <= C)
  __device__ __forceinline__ void issue_loads(const StoreDesc &sd, int n_, int base_) {
    if (BIG) return;
    // (broadcasts from lane 0: tells the compiler the operands of the bulk copies are warp-uniform)
    n_ = __shfl_sync(0xffffffffu, n_, 0);
    base_ = __shfl_sync(0xffffffffu, base_, 0);
    loads_armed = n_ > 0 && n_ <= C;
    if (loads_armed && lane == 0) {
      const unsigned bytes = (unsigned)((n_ + 3) & ~3) * 4u;
      mbar_expect_tx(bar, bytes * (unsigned)ncol);
      if (XC) {
        for (int c = 0; c < ncol; c++) bulk_g2s(buf + c * C, sd.col[c] + base_, bytes, bar);
      } else {
#pragma unroll
        for (int c = 0; c < NREC; c++) bulk_g2s(buf + c * C, sd.col[c] + base_, bytes, bar);
      }
    }
  }

  // key of the cell that reaches cell (lx, ly, lz) of this tile by a move in this lane's direction
  template <class TG>
  __device__ __forceinline__ int source_key(const TG &tg, int dc, int lx, int ly, int lz) const {
    // the direction this lane looks at when a cell collects its arrivals: lane = direction code
    // (recomputed here: a lane constant kept across the particle loop costs registers)
    int sx, sy, sz;
    dir_decode<D3>(dc, sx, sy, sz);
    int qx = lx - sx, qy = ly - sy, qz = lz - sz;
    const int tx = D3 ? (qx < 0 ? -1 : (qx >= tg.bs[0] ? 1 : 0)) : 0;
    const int ty = qy < 0 ? -1 : (qy >= tg.bs[1] ? 1 : 0);
    const int tz = qz < 0 ? -1 : (qz >= tg.bs[2] ? 1 : 0);
    qx -= tx * tg.bs[0];
    qy -= ty * tg.bs[1];
    qz -= tz * tg.bs[2];
    return nbt[(tz + 1) * 9 + (ty + 1) * 3 + (tx + 1)] + (qz * tg.bs[1] + qy) * tg.bs[0] + qx;
  }

  // The header word this lane needs to find the arrivals of cell ci of the tile (its neighbour in
  // this lane's direction, that direction's mask): requested one cell ahead of begin_cell().
  template <class TG>
  __device__ __forceinline__ unsigned fetch_mask(const StoreDesc &sd, const TG &tg, int ci, int &src) const {
    src = 0;
    const int dc = keep_in_loop(lane);  // lane = direction code
    if (!(dc < ND && dc != STAY) || ci >= tg.cpb) return 0u;
    const int lx = ci % tg.bs[0], t = ci / tg.bs[0];
    src = source_key(tg, dc, lx, t % tg.bs[1], t / tg.bs[1]);
    return sd.xin.mask[(size_t)src * XW + dc];
  }

  // writes the arrival-list window [a0, a0 + WALK_AC): entry = direction lane << 8 | record index
  __device__ __forceinline__ void fill_window(unsigned mask) {
    int g = my_start - a0;
    while (mask) {
      const int j = __ffs(mask) - 1;
      if (g >= 0 && g < WALK_AC) arr[g] = (uint16_t)((lane << 8) | j);
      g++;
      mask &= mask - 1;
    }
    __syncwarp();
  }

  // Start of a cell: its arrivals (from the neighbours' header words), whether it fits the image;
  // waits for its resident run.
  __device__ __forceinline__ void begin_cell(int key_, int n_, int base_, int cap_, unsigned mask, int src) {
    key = key_;
    n = n_;
    base = base_;
    cap = cap_;
    const int cntm = __popc(mask);
    my_mask = mask;
    my_src = src;
    if (BIG) {  // the global path walks the arrivals through a list in shared memory
      nbk[lane] = src;
      int inc = cntm;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
      }
      na = __shfl_sync(0xffffffffu, inc, 31);
      my_start = inc - cntm;
      a0 = 0;
      if (na) fill_window(mask);
    } else {
      na = __reduce_add_sync(0xffffffffu, cntm);
    }
    fits = n + na <= C;
    nh = 0;
    tcur = 0;
    nleave = 0;
    if (!BIG && loads_armed) {
      mbar_wait(bar, parity);
      parity ^= 1;
      loads_armed = false;
    }
  }

  // ---- image path ---------------------------------------------------------------------------------

  // The arrivals' record words go to the image slots [n, n + na) behind the residents, by
  // asynchronous 4-byte copies, a lane per arrival.  Which record a slot takes is first noted in
  // the slot itself (the lane that looked at a neighbour's header writes "my direction, record j"
  // for every record it found; a shared counter hands out the slots: the order of arrivals inside
  // a cell is immaterial).  Wait with arrivals_landed().
  __device__ __forceinline__ void stage_arrivals(const StoreDesc &sd) {
    int *note = reinterpret_cast<int *>(buf) + (NREC - 1) * C + n;  // the species column's tail
    unsigned m = my_mask;
    if (m) {
      int a = atomicAdd(acnt, __popc(m));
      while (m) {
        note[a++] = (lane << 8) | (__ffs(m) - 1);
        m &= m - 1;
      }
    }
    __syncwarp();
    if (lane == 0) *acnt = 0;
    for (int a0_ = 0; a0_ < na; a0_ += 32) {
      const int a = a0_ + lane;
      const int e = a < na ? note[a] : 0;
      const int src = __shfl_sync(0xffffffffu, my_src, (e >> 8) & 31);
      if (a < na) {
        const size_t idx = (size_t)src * PSC_XCAP + (e & 255);
        const float *r = reinterpret_cast<const float *>(sd.xin.rec + idx);
        float *q = buf + n + a;
#pragma unroll
        for (int w = 0; w < NREC; w++) cp_async4(q + w * C, r + w, true);
        if (XC) {
          if (sd.icol_x2d >= 0) cp_async4(q + sd.icol_x2d * C, r + 7, true);
          if (sd.icol_id >= 0) cp_async4(q + sd.icol_id * C, sd.xin.id + idx, true);
        }
      }
    }
    cp_async_commit();
  }
  // Before the first chunk that touches slots >= n: the arrivals are in the image, and the slots
  // between the last particle and the end of its chunk hold a harmless particle (at rest, no
  // charge) instead of whatever the copies left there.
  __device__ __forceinline__ void arrivals_landed() {
    cp_async_wait<0>();
    const int T = n + na;
    const int s = T + lane;
    if (s < ((T + 31) & ~31)) {
      float *q = buf + s;
#pragma unroll
      for (int c = 0; c < NREC; c++) q[c * C] = (c < (D3 ? 3 : 2)) ? 0.25f : 0.f;
    }
    __syncwarp();
  }

  // particle v of the image, no bounds check
  __device__ __forceinline__ void load_image(int v, Part &p) const {
    const float *q = buf + v;
    if (D3) {
      p.ax = q[0]; p.ay = q[C]; p.az = q[2 * C]; p.ux = q[3 * C]; p.uy = q[4 * C]; p.uz = q[5 * C];
      p.qw = q[6 * C]; p.sp = __float_as_int(q[7 * C]);
    } else {
      p.ax = 0.f;
      p.ay = q[0]; p.az = q[C]; p.ux = q[2 * C]; p.uy = q[3 * C]; p.uz = q[4 * C];
      p.qw = q[5 * C]; p.sp = __float_as_int(q[6 * C]);
    }
  }

  // Files particle v0 + lane of the image after its push: the momentum always, the offsets only if
  // it stays; a leaver keeps its old offsets and is noted as a hole (see leaver()).
  __device__ __forceinline__ void store_image(int v0, bool act, bool leave, const Part &pn) {
    const int v = v0 + lane;
    const unsigned mrl = __ballot_sync(0xffffffffu, act && leave);
    if (act) {
      float *q = buf + v;
      if (D3) {
        if (!leave) { q[0] = pn.ax; q[C] = pn.ay; q[2 * C] = pn.az; }
        q[3 * C] = pn.ux; q[4 * C] = pn.uy; q[5 * C] = pn.uz;
      } else {
        if (!leave) { q[0] = pn.ay; q[C] = pn.az; }
        q[2 * C] = pn.ux; q[3 * C] = pn.uy; q[4 * C] = pn.uz;
      }
      if (leave) {
        const int hi = nh + __popc(mrl & ((1u << lane) - 1u));  // (not the lanemask register: an S2R per chunk)
        if (hi < WALK_HC) holes[hi] = (uint8_t)v;
      }
    }
    if (lane == 0) hbm[v0 >> 5] = mrl;
    nh += __popc(mrl);
  }

  // slot of the i-th hole (ascending): from the byte list, beyond it from the bitmap
  __device__ __forceinline__ int hole_at(int i) const {
    if (i < WALK_HC) return holes[i];
    int acc = 0;
    for (int w = 0; w < 8; w++) {
      const unsigned m = hbm[w];
      const int c = __popc(m);
      if (i < acc + c) return w * 32 + (int)__fns(m, 0, i - acc + 1);
      acc += c;
    }
    return 0;
  }

  // leaver i of the hole list: its image values (OLD offsets, NEW momentum) and optional columns
  __device__ __forceinline__ void leaver(const StoreDesc &sd, int i, Part &p, float &x2d, int &id) const {
    const int h = hole_at(i);
    load_image(h, p);
    x2d = 0.f;
    id = 0;
    if (XC) {
      if (sd.icol_x2d >= 0) x2d = buf[sd.icol_x2d * C + h];
      if (sd.icol_id >= 0) id = __float_as_int(buf[sd.icol_id * C + h]);
    }
  }

  // End of a cell on the image path: close the holes from the tail of the image, write the image's
  // dynamic columns back, the static ones where a particle is new in its slot; publish the count
  // and the exchange row; start fetching the next cell (next_n <= 0: none).
  __device__ __forceinline__ void end_image(const StoreDesc &sd, int next_n, int next_base) {
    __syncwarp();
    const int T = n + na;
    int newcnt = T - nh;
    if (nh > 0) {
      int done = 0;
      for (int t0 = newcnt; t0 < T; t0 += 32) {
        const int s = t0 + lane;
        const bool valid = s < T && !((hbm[s >> 5] >> (s & 31)) & 1u);
        const unsigned mv = __ballot_sync(0xffffffffu, valid);
        if (valid) {
          const int h = hole_at(done + __popc(mv & lt));  // ascending: the first holes are < newcnt
          for (int c = 0; c < ncol; c++) buf[c * C + h] = buf[c * C + s];
          if (h < n)
            for (int c = NDYN; c < ncol; c++) st_stream(sd.col[c] + (size_t)base + h, buf[c * C + s]);
        }
        done += __popc(mv);
      }
      __syncwarp();
    }
    if (newcnt > cap) {  // no room for all arrivals: the excess spills (and forces a re-layout)
      for (int s = cap + lane; s < newcnt; s += 32) {
        float w[8];
#pragma unroll
        for (int c = 0; c < NREC; c++) w[c] = buf[c * C + s];
        if (!D3) w[7] = (XC && sd.icol_x2d >= 0) ? buf[sd.icol_x2d * C + s] : 0.f;
        spill_particle(sd, key, w, (XC && sd.icol_id >= 0) ? __float_as_int(buf[sd.icol_id * C + s]) : 0);
      }
      newcnt = cap;
    }
    // arrivals that ended up behind the old residents: their static columns are new in global memory
    for (int s = n + lane; s < newcnt; s += 32)
      for (int c = NDYN; c < ncol; c++) st_stream(sd.col[c] + (size_t)base + s, buf[c * C + s]);
    fence_proxy_async();
    __syncwarp();
    {
      const int cnt_u = __shfl_sync(0xffffffffu, newcnt, 0), base_u = __shfl_sync(0xffffffffu, base, 0);
      if (lane == 0 && cnt_u > 0) {
        const unsigned bytes = (unsigned)((cnt_u + 3) & ~3) * 4u;
#pragma unroll
        for (int c = 0; c < NDYN; c++) bulk_s2g(sd.col[c] + base_u, buf + c * C, bytes);
        bulk_commit();
      }
    }
    publish(sd, newcnt);
    if (lane == 0) bulk_wait_read0();  // the image may be overwritten once the copy engine has read it
    __syncwarp();
    if (next_n > 0) issue_loads(sd, next_n, next_base);
  }

  // a cell this launch leaves to the other one: nothing changes, only the next fetch starts
  __device__ __forceinline__ void skip_cell(const StoreDesc &sd, int next_n, int next_base) {
    if (next_n > 0) issue_loads(sd, next_n, next_base);
  }

  __device__ __forceinline__ void publish(const StoreDesc &sd, int newcnt) {
    if (lane == 0) {
      sd.cnt[key] = newcnt;
      // a cell that has outgrown every cell the host knows of reports its size: the per-warp image
      // of the kernels follows the largest cell at the host's next look at the status block
      if (newcnt > sd.maxcnt_known) atomicMax(sd.maxcnt, (uint32_t)newcnt);
    }
    if (lane < XW) sd.xout.mask[(size_t)key * XW + lane] = xrow[lane];
    __syncwarp();
    if (lane < XW) xrow[lane] = 0u;
  }

  // ---- records ------------------------------------------------------------------------------------

  // the 8 record words of a particle (positions as given)
  __device__ __forceinline__ static void to_words(float (&w)[8], const Part &p, float x2d) {
    if (D3) {
      w[0] = p.ax; w[1] = p.ay; w[2] = p.az; w[3] = p.ux; w[4] = p.uy; w[5] = p.uz; w[6] = p.qw;
      w[7] = __int_as_float(p.sp);
    } else {
      w[0] = p.ay; w[1] = p.az; w[2] = p.ux; w[3] = p.uy; w[4] = p.uz; w[5] = p.qw;
      w[6] = __int_as_float(p.sp); w[7] = x2d;
    }
  }

  // writes record xi of the current cell's row (moved by direction code dc; positions relative
  // to the destination cell), or spills it if the row is full
  __device__ __forceinline__ void emit(const StoreDesc &sd, int xi, int dc, const float (&w)[8], int id,
                                       int dest_key) {
    if (xi < PSC_XCAP) {
      atomicOr(&xrow[dc], 1u << xi);
      const size_t idx = (size_t)key * PSC_XCAP + xi;
      XRec r;
      r.a = make_uint4(__float_as_uint(w[0]), __float_as_uint(w[1]), __float_as_uint(w[2]), __float_as_uint(w[3]));
      r.b = make_uint4(__float_as_uint(w[4]), __float_as_uint(w[5]), __float_as_uint(w[6]), __float_as_uint(w[7]));
      sd.xout.rec[idx] = r;
      if (XC && sd.xout.id) sd.xout.id[idx] = id;
    } else {
      spill_particle(sd, dest_key, w, id);
    }
  }

  // ---- global path (BIG) --------------------------------------------------------------------------

  // Loads particle v0 + lane of the cell (residents from the columns, then arrivals from the
  // neighbours' rows).  Returns whether the lane holds a particle.
  __device__ __forceinline__ bool load_global(const StoreDesc &sd, int v0, Part &p, float &x2d, int &id) {
    const int v = v0 + lane;
    const bool act = v < n + na;
    p.ax = p.ay = p.az = 0.25f;
    p.ux = p.uy = p.uz = p.qw = 0.f;
    p.sp = 0;
    x2d = 0.f;
    id = 0;
    if (v0 + 32 > n && na) {  // warp-uniform: this chunk contains arrivals
      if (v0 + 32 - n > a0 + WALK_AC) {  // next window of the arrival list
        a0 = v0 > n ? v0 - n : 0;
        const bool have = lane < ND && lane != STAY;
        const unsigned mask = have ? sd.xin.mask[(size_t)nbk[lane] * XW + lane] : 0u;
        __syncwarp();
        fill_window(mask);
      }
      if (act && v >= n) {
        const int e = arr[v - n - a0];
        const size_t idx = (size_t)nbk[e >> 8] * PSC_XCAP + (e & 255);
        const XRec r = sd.xin.rec[idx];
        if (D3) {
          p.ax = __uint_as_float(r.a.x); p.ay = __uint_as_float(r.a.y); p.az = __uint_as_float(r.a.z);
          p.ux = __uint_as_float(r.a.w); p.uy = __uint_as_float(r.b.x); p.uz = __uint_as_float(r.b.y);
          p.qw = __uint_as_float(r.b.z); p.sp = (int)r.b.w;
        } else {
          p.ay = __uint_as_float(r.a.x); p.az = __uint_as_float(r.a.y);
          p.ux = __uint_as_float(r.a.z); p.uy = __uint_as_float(r.a.w); p.uz = __uint_as_float(r.b.x);
          p.qw = __uint_as_float(r.b.y); p.sp = (int)r.b.z; x2d = __uint_as_float(r.b.w);
        }
        if (XC && sd.xin.id) id = sd.xin.id[idx];
      }
    }
    if (act && v < n) {
      const size_t s = (size_t)base + v;
      if (D3) {
        p.ax = ld_stream(sd.col[0] + s); p.ay = ld_stream(sd.col[1] + s); p.az = ld_stream(sd.col[2] + s);
        p.ux = ld_stream(sd.col[3] + s); p.uy = ld_stream(sd.col[4] + s); p.uz = ld_stream(sd.col[5] + s);
        p.qw = ld_stream(sd.col[6] + s); p.sp = __float_as_int(ld_stream(sd.col[7] + s));
      } else {
        p.ay = ld_stream(sd.col[0] + s); p.az = ld_stream(sd.col[1] + s);
        p.ux = ld_stream(sd.col[2] + s); p.uy = ld_stream(sd.col[3] + s); p.uz = ld_stream(sd.col[4] + s);
        p.qw = ld_stream(sd.col[5] + s); p.sp = __float_as_int(ld_stream(sd.col[6] + s));
      }
      if (XC) {
        if (sd.icol_x2d >= 0) x2d = ld_stream(sd.col[sd.icol_x2d] + s);
        if (sd.icol_id >= 0) id = __float_as_int(ld_stream(sd.col[sd.icol_id] + s));
      }
    }
    return act;
  }

  // index of the next leaver's record in the cell's exchange row (all lanes)
  __device__ __forceinline__ int leaver_slot(bool leave) {
    const unsigned m = __ballot_sync(0xffffffffu, leave);
    const int xi = nleave + __popc(m & lt);
    nleave += __popc(m);
    return xi;
  }

  // every particle of the chunk that stays is compacted to the front of the cell, in place (the
  // write cursor tcur never passes the reads); pn: the new values
  __device__ __forceinline__ void store_global(const StoreDesc &sd, bool stay, const Part &pn, float x2d, int id) {
    const unsigned ms = __ballot_sync(0xffffffffu, stay);
    const int slot = tcur + __popc(ms & lt);
    __syncwarp();
    if (stay) {
      float w[8];
      to_words(w, pn, x2d);
      if (slot < cap) {
        const size_t s = (size_t)base + slot;
#pragma unroll
        for (int c = 0; c < NREC; c++) st_stream(sd.col[c] + s, w[c]);
        if (XC) {
          if (sd.icol_x2d >= 0) st_stream(sd.col[sd.icol_x2d] + s, x2d);
          if (sd.icol_id >= 0) st_stream(sd.col[sd.icol_id] + s, __int_as_float(id));
        }
      } else {
        spill_particle(sd, key, w, id);
      }
    }
    tcur += __popc(ms);
  }

  __device__ __forceinline__ void end_global(const StoreDesc &sd) {
    __syncwarp();
    publish(sd, tcur < cap ? tcur : cap);
  }

  __device__ __forceinline__ void finish() {
    if (!BIG && lane == 0) bulk_wait_all();
    __syncwarp();
  }
};
#undef C
