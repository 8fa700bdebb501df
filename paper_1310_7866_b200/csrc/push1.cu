// push1.cu -- the fused particle loop of Fig. 8 for first-order
// particles: gather E,B with b1 weights (Eq. 11, 29-31), Boris push (Eq. 27-28),
// move (Eq. 26), Villasenor-Buneman charge-conserving deposit, periodic wrap.
//
// One thread block per sort block ("supercell"): the block stages the E/B values
// its cells can touch (tile + 1 halo point each side) in shared memory and accumulates current
// in a shared J tile (tile + 1 low / 2 high halo nodes) that is flushed to global J once.  A
// warp takes one CELL at a time and walks that cell's slots in chunks of 32, so the cell -- and
// with it every tile address that does not depend on the in-cell offset -- is warp-uniform: the
// gather becomes the evaluation of per-cell polynomials (the warp turns the cell's field stencil
// into a small coefficient table once per cell, "per-cell gather tables" below), and the currents
// of the trajectories that stay inside the cell (the great majority) are summed in registers
// over the whole cell and reduced across the warp once per cell.
//
// This is the single particle loop of PAPER.md:603 ("only one loop each time step that reads
// and writes all particle data"), over the cell store of store.cuh: a cell's resident particles
// arrive in shared memory through one bulk asynchronous copy per column, are advanced there in
// place and written back the same way; the few that leave go, as 32-byte records tagged with the
// direction code of their move, into the cell's exchange row, from which the destination cell's
// warp collects them in the NEXT push (reorder on load).  There is no sort pass between pushes.
//
// Positions are in the internal form (include/psc.h): in-cell offset a in [0,1) per direction;
// the cell is implied by the segment.  The move is b = a + v dt/dx; a particle that leaves its
// cell (b < 0 or b >= 1; at most one cell per direction) is recorded with offset
// b -/+ 1 and the direction code of the move; the destination's warp turns code + source cell
// back into "mine" with the periodic wrap -- the single-GPU form of the particle exchange
// (PAPER.md:403).  No floor(), no float->int conversion and no absolute coordinate appear here.
//
// The VB current is the exact flux of a b0-shaped cloud moving on the straight line
// x^{n+1/2} -> x^{n+3/2}; it is evaluated by splitting the line at the cell faces it crosses
// (at most one per direction because dt <= dx/2).  For a segment a -> b inside one cell, with
// m = (a+b)/2 and del = b-a in units of cells:
//   j_c(c+1/2, e+al, f+be) += (qw/dV)(del_c dx_c/dt) W_{al,be},
//   W_00 = (1-m_e)(1-m_f) + del_e del_f/12, W_10 = m_e(1-m_f) - ..., W_01 = (1-m_e)m_f - ...,
//   W_11 = m_e m_f + del_e del_f/12;
// in 2-d (x invariant) the in-plane weights reduce to {1-m, m} and the out-of-plane current is
// the time average of v_x S_y S_z over the segment (A12).
#include "store.cuh"

#ifndef PSC_MINB2D
#define PSC_MINB2D 6  // blocks per SM of the default 2-d kernel
#endif
#ifndef PSC_THREADS2D
#define PSC_THREADS2D 128  // threads per block of the default 2-d kernel
#endif
#ifndef PSC_MINB3D
#define PSC_MINB3D 5  // ... of the default 3-d kernel
#endif
namespace {

// per-warp queue of trajectories that leave their cell: 2-d (3 % leavers; shared memory decides
// the blocks per SM) 24 entries, walked 16-24 at a time; 3-d (12 % leavers) 64, walked 32 at a time
template <bool D3> struct QCap { static constexpr int v = D3 ? 64 : 24; };
// rows of a queue entry: 0 packed cell (lx | ly << 10 | lz << 20), 1 ax, 2 ay, 3 az, 4 endx (2-d: v_x),
// 5 endy, 6 endz, 7 qw
constexpr int QROWS2 = 7, QROWS3 = 8;


// Tile geometry.  CBS != 0: the sort block is CBS cells along every active direction (the
// library defaults, 8x8 in 2-d and 4x4x4 in 3-d), known at compile time so that every tile
// extent, stride and shared-memory offset folds into an immediate; CBS == 0: run-time block.
// TM: the tiles are staged by TMA tensor copies (3-d default block only), whose boxes must be a
// multiple of 16 bytes along x: the field tile is 8 x 6 x 6 instead of 6 x 6 x 6, the J tile
// 8 x 7 x 7 instead of 7 x 7 x 7 (the extra points are loaded / stay zero and are never used).
template <bool D3, int CBS, bool TM = false>
struct TileGeom {
  int o[3];        // first cell of the tile (global cell coordinates)
  int bs[3], cpb;  // block size in cells, cells per block
  int fe[3], fvol; // field tile extents (bs+2 | 1), volume
  int je[3], jvol; // J tile extents (bs+3 | 1), volume
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
    fe[0] = TM ? 8 : (D3 ? bs[0] + 2 : 1);
    fe[1] = bs[1] + 2;
    fe[2] = bs[2] + 2;
    je[0] = TM ? 8 : (D3 ? bs[0] + 3 : 1);
    je[1] = bs[1] + 3;
    je[2] = bs[2] + 3;
    fvol = fe[0] * fe[1] * fe[2];
    jvol = je[0] * je[1] * je[2];
  }
};

// ---- warp-level reduction of the home-cell currents -------------------------------------------
// The particle list is cell-ordered, so the 32 lanes of a warp mostly sit in ONE cell and their
// first trajectory segment deposits onto the same 8 (2-d) / 12 (3-d) J points.  Summing those in
// registers and issuing one shared-memory add per point per warp replaces 32-way conflicting
// atomics (shared fp32 atomicAdd is a compare-and-swap loop on sm_100a: ATOMS.CAST.SPIN) by
// shuffles.  The reduction halves the number of live values at every butterfly stage
// ("transpose-reduce"): 9 shuffles for 8 values, 13 for 12, instead of 5 per value.

__device__ __forceinline__ float xadd(bool up, float lo, float hi, int m) {
  // lanes with `up` keep hi and hand lo to their partner; the others keep lo and hand over hi
  return (up ? hi : lo) + __shfl_xor_sync(0xffffffffu, up ? lo : hi, m);
}

// returns, in every lane, the warp total of v[(lane >> 2) & 7]
__device__ __forceinline__ float warp_reduce8(const float (&v)[8], int lane) {
  const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
  float w[4], u[2];
#pragma unroll
  for (int i = 0; i < 4; i++) w[i] = xadd(b4, v[i], v[i + 4], 16);
#pragma unroll
  for (int i = 0; i < 2; i++) u[i] = xadd(b3, w[i], w[i + 2], 8);
  float t = xadd(b2, u[0], u[1], 4);
  t += __shfl_xor_sync(0xffffffffu, t, 2);
  t += __shfl_xor_sync(0xffffffffu, t, 1);
  return t;
}

// returns the warp total of v[red12_index(lane)]
__device__ __forceinline__ int red12_index(int lane) {
  return ((lane & 16) ? 6 : 0) + ((lane & 8) ? 3 : 0) + ((lane & 2) ? 2 : ((lane & 4) ? 1 : 0));
}
__device__ __forceinline__ float warp_reduce12(const float (&v)[12], int lane) {
  const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4, b1 = lane & 2;
  float w[6], u[3];
#pragma unroll
  for (int i = 0; i < 6; i++) w[i] = xadd(b4, v[i], v[i + 6], 16);
#pragma unroll
  for (int i = 0; i < 3; i++) u[i] = xadd(b3, w[i], w[i + 3], 8);
  const float t0 = xadd(b2, u[0], u[1], 4);
  const float t1 = u[2] + __shfl_xor_sync(0xffffffffu, u[2], 4);
  float r = xadd(b1, t0, t1, 2);
  r += __shfl_xor_sync(0xffffffffu, r, 1);
  return r;
}

// in-cell VB currents of one segment a -> b (both in the coordinates of the segment's cell), in
// the order the reductions and the per-lane J offsets use:
//   3-d: jx{(y,z),(y+1,z),(y,z+1),(y+1,z+1)}  jy{(z,x),(z+1,x),(z,x+1),(z+1,x+1)}
//        jz{(x,y),(x+1,y),(x,y+1),(x+1,y+1)}
//   2-d: jx{(y,z),(y+1,z),(y,z+1),(y+1,z+1)}  jy{z,z+1}  jz{y,y+1}
template <bool D3>
__device__ __forceinline__ void vb_values(float (&v)[D3 ? 12 : 8], float ax, float ay, float az,
                                          float bx, float by, float bz, float tau, float fx,
                                          float fy, float fz, float qvx) {
  const float my = 0.5f * (ay + by), mz = 0.5f * (az + bz);
  const float dy = by - ay, dz = bz - az;
  if (D3) {
    const float mx = 0.5f * (ax + bx), dx = bx - ax;
    {
      const float c = fx * dx, h = dy * dz * (1.0f / 12.0f);
      v[0] = c * ((1.f - my) * (1.f - mz) + h);
      v[1] = c * (my * (1.f - mz) - h);
      v[2] = c * ((1.f - my) * mz - h);
      v[3] = c * (my * mz + h);
    }
    {
      const float c = fy * dy, h = dz * dx * (1.0f / 12.0f);
      v[4] = c * ((1.f - mz) * (1.f - mx) + h);
      v[5] = c * (mz * (1.f - mx) - h);
      v[6] = c * ((1.f - mz) * mx - h);
      v[7] = c * (mz * mx + h);
    }
    {
      const float c = fz * dz, h = dx * dy * (1.0f / 12.0f);
      v[8] = c * ((1.f - mx) * (1.f - my) + h);
      v[9] = c * (mx * (1.f - my) - h);
      v[10] = c * ((1.f - mx) * my - h);
      v[11] = c * (mx * my + h);
    }
  } else {
    {
      const float c = qvx * tau, h = dy * dz * (1.0f / 12.0f);
      v[0] = c * ((1.f - my) * (1.f - mz) + h);
      v[1] = c * (my * (1.f - mz) - h);
      v[2] = c * ((1.f - my) * mz - h);
      v[3] = c * (my * mz + h);
    }
    {
      const float c = fy * dy;
      v[4] = c * (1.f - mz);
      v[5] = c * mz;
    }
    {
      const float c = fz * dz;
      v[6] = c * (1.f - my);
      v[7] = c * my;
    }
  }
}

// The same in-cell currents, accumulated as MOMENTS: with e, f the two transverse midpoints of a
// component and c its prefactor, the four values are c((1-e)(1-f)+h), c(e(1-f)-h), c((1-e)f-h),
// c(ef+h), i.e. linear in M0 = c, M1 = c e, M2 = c f, M3 = c (e f + h):
//   v_a = M0 - M1 - M2 + M3, v_b = M1 - M3, v_c = M2 - M3, v_d = M3
// (2-d in-plane components: c(1-m), c m from N0 = c, N1 = c m).  Summing the moments over a
// cell's particles and converting once per cell (moments_to_values) costs 7 instead of 16
// operations per particle and component.  acc uses the slots of the values it turns into.
template <bool D3>
__device__ __forceinline__ void vb_moments(float (&acc)[D3 ? 12 : 8], float ax, float ay, float az,
                                           float bx, float by, float bz, float fx, float fy,
                                           float fz, float qvx) {
  const float my = 0.5f * (ay + by), mz = 0.5f * (az + bz);
  const float dy = by - ay, dz = bz - az;
  auto add4 = [](float *m, float c, float e, float f, float dd) {
    m[0] += c;
    m[1] = fmaf(c, e, m[1]);
    m[2] = fmaf(c, f, m[2]);
    m[3] = fmaf(c, fmaf(e, f, dd * (1.0f / 12.0f)), m[3]);
  };
  if (D3) {
    const float mx = 0.5f * (ax + bx), dx = bx - ax;
    add4(acc + 0, fx * dx, my, mz, dy * dz);
    add4(acc + 4, fy * dy, mz, mx, dz * dx);
    add4(acc + 8, fz * dz, mx, my, dx * dy);
  } else {
    add4(acc + 0, qvx, my, mz, dy * dz);
    const float cy = fy * dy, cz = fz * dz;
    acc[4] += cy;
    acc[5] = fmaf(cy, mz, acc[5]);
    acc[6] += cz;
    acc[7] = fmaf(cz, my, acc[7]);
  }
}

template <bool D3>
__device__ __forceinline__ void moments_to_values(float (&acc)[D3 ? 12 : 8]) {
#pragma unroll
  for (int b = 0; b < (D3 ? 12 : 4); b += 4) {
    const float m0 = acc[b], m1 = acc[b + 1], m2 = acc[b + 2], m3 = acc[b + 3];
    acc[b] = (m0 - m1) - (m2 - m3);
    acc[b + 1] = m1 - m3;
    acc[b + 2] = m2 - m3;
  }
  if (!D3) {
    acc[4] -= acc[5];
    acc[6] -= acc[7];
  }
}

// Walks the straight line a -> end (cells; at most one face crossing per direction because
// dt <= dx/2) and deposits every segment -- the slow path of the kernel below,
// taken by the trajectories that leave their cell.
// The segments' currents go straight to the global J with fire-and-forget reductions (RED.ADD.F32,
// resolved in the L2, where J lives): a shared-memory fp32 atomicAdd is a compare-and-swap loop on
// sm_100a whose retries -- the trajectories drained together come from a few cells and hit the
// same points -- made this path the largest single stall of the kernel.  (lx, ly, lz): the
// trajectory's cell inside the tile; gnode0: global index of the tile's first cell's node; rel:
// the NV point offsets of vb_values in the global array.
template <bool D3, class TG>
__device__ __forceinline__ void vb_walk(float *__restrict__ J, const GridDesc &gd, int gnode0, int lx,
                                        int ly, int lz, float ax, float ay, float az, float endx,
                                        float endy, float endz, float fx, float fy, float fz,
                                        float qvx, const int *__restrict__ rel) {
  constexpr int NV = D3 ? 12 : 8;
  const float ddx = endx - ax, ddy = endy - ay, ddz = endz - az;
  const int sxd = D3 ? (endx >= 1.f ? 1 : (endx < 0.f ? -1 : 0)) : 0;
  const int syd = endy >= 1.f ? 1 : (endy < 0.f ? -1 : 0);
  const int szd = endz >= 1.f ? 1 : (endz < 0.f ? -1 : 0);
  float tx = sxd ? ((sxd > 0 ? 1.f - ax : -ax) / ddx) : 2.f;
  float ty = syd ? ((syd > 0 ? 1.f - ay : -ay) / ddy) : 2.f;
  float tz = szd ? ((szd > 0 ? 1.f - az : -az) / ddz) : 2.f;
  float px = ax, py = ay, pz = az;  // segment start, in origin-cell coordinates
  int rx = 0, ry = 0, rz = 0;       // current cell relative to the origin cell
  float tprev = 0.f;
#pragma unroll 1
  for (int seg = 0; seg < (D3 ? 4 : 3); seg++) {
    const float t = fminf(fminf(tx, ty), fminf(tz, 1.f));
    const int which = (t >= 1.f) ? 3 : (tx <= ty && tx <= tz) ? 0 : (ty <= tz ? 1 : 2);
    float qx = ax + t * ddx, qy = ay + t * ddy, qz = az + t * ddz;  // segment end
    if (which == 3) {
      qx = endx; qy = endy; qz = endz;
    } else if (which == 0) {
      qx = sxd > 0 ? (float)(rx + 1) : (float)rx;
    } else if (which == 1) {
      qy = syd > 0 ? (float)(ry + 1) : (float)ry;
    } else {
      qz = szd > 0 ? (float)(rz + 1) : (float)rz;
    }
    {
      float v[NV];
      vb_values<D3>(v, px - rx, py - ry, pz - rz, qx - rx, qy - ry, qz - rz, t - tprev, fx, fy, fz, qvx);
      float *node = J + gnode0 + (D3 ? (lx + rx) : 0) + (ly + ry) * gd.st[1] + (lz + rz) * gd.st[2];
#pragma unroll
      for (int i = 0; i < NV; i++) atomicAdd(node + rel[i], v[i]);
    }
    if (which == 3) break;
    if (which == 0) { rx += sxd; tx = 2.f; }
    else if (which == 1) { ry += syd; ty = 2.f; }
    else { rz += szd; tz = 2.f; }
    px = qx; py = qy; pz = qz;
    tprev = t;
  }
}

// Drains n (<= 32) queue entries starting at `start`: deposits every segment of each trajectory.
template <bool D3, class TG>
__device__ __forceinline__ void drain_queue(float *__restrict__ J, const TG &tg, const GridDesc &gd,
                                            int gnode0, const float *__restrict__ q,
                                            const int *__restrict__ rel, int start, int n, int lane) {
  constexpr int QCAP = QCap<D3>::v;
  if (lane < n) {
    const int e = start + lane;
    const int packed = __float_as_int(q[0 * QCAP + e]);
    const float ax = D3 ? q[1 * QCAP + e] : 0.f, ay = q[2 * QCAP + e], az = q[3 * QCAP + e];
    const float ex = q[4 * QCAP + e], ey = q[5 * QCAP + e], ez = q[6 * QCAP + e];
    const float qw = q[(D3 ? 7 : 1) * QCAP + e];
    const int lx = packed & 1023, ly = (packed >> 10) & 1023, lz = packed >> 20;
    // 2-d: the endx slot carries v_x: the out-of-plane current needs the velocity
    const float fx = qw * gd.cur[0], fy = qw * gd.cur[1], fz = qw * gd.cur[2];
    const float qvx = D3 ? 0.f : qw * gd.inv_dV * ex;
    vb_walk<D3, TG>(J, gd, gnode0, lx, ly, lz, D3 ? ax : 0.f, ay, az, D3 ? ex : 0.f, ey, ez, fx, fy, fz,
                    qvx, rel);
  }
  __syncwarp();
}

// ---- per-cell gather tables ------------------------------------------------------------------
// Inside one cell the b1-weighted value of a field component (Eq. 11) is a
// multilinear polynomial of the in-cell offsets a: along a direction in which the component sits
// on the nodes the two stencil points are l, l+1 with weight a; along a direction in which it is
// half-staggered they are l-1, l with weight a + 1/2 (a < 1/2) or l, l+1 with weight a - 1/2
// (a >= 1/2) -- two PIECES.  So a component has 1, 2 or 4 pieces per cell (2-d: 13 in all, 3-d:
// 18), each with 4 (2-d) / 8 (3-d) polynomial coefficients.  The warp that owns a cell computes
// them once per cell (a lane per piece, from the block's field tile) into a small per-warp table;
// a particle then needs one (two) 16-byte shared loads and 3 (7) FMAs per component instead of
// 4 (8) loads and 5 (14) operations.
template <bool D3> struct GTab {
  static constexpr int NP = D3 ? 18 : 13;  // pieces
  static constexpr int W = D3 ? 8 : 4;     // coefficients per piece
  static constexpr int FLOATS = NP * W;
};

// What lane `l` (a piece) reads and how it shifts: off = offset of its base stencil point from
// the cell's node in the field tile, sg* = weight shift (0 node-centred, +1/2 lower piece, -1/2
// upper piece).  Piece order: Ex[hx] Ey[hy] Ez[hz] Bx[hy + 2 hz] By[hx + 2 hz] Bz[hx + 2 hy]
// (2-d: no hx: Ex, Ey[hy], Ez[hz], Bx[hy + 2 hz], By[hz], Bz[hy]).
template <bool D3>
__device__ __forceinline__ void piece_desc(int l, int fs1, int fs2, int fvol, int &off, float &sgx,
                                           float &sgy, float &sgz) {
  int comp, hx = -1, hy = -1, hz = -1;  // -1: node-centred along that direction
  if (D3) {
    if (l < 2) { comp = 0; hx = l; }
    else if (l < 4) { comp = 1; hy = l - 2; }
    else if (l < 6) { comp = 2; hz = l - 4; }
    else if (l < 10) { comp = 3; hy = (l - 6) & 1; hz = (l - 6) >> 1; }
    else if (l < 14) { comp = 4; hx = (l - 10) & 1; hz = (l - 10) >> 1; }
    else { comp = 5; hx = (l - 14) & 1; hy = ((l - 14) >> 1) & 1; }
  } else {
    if (l < 1) { comp = 0; }
    else if (l < 3) { comp = 1; hy = l - 1; }
    else if (l < 5) { comp = 2; hz = l - 3; }
    else if (l < 9) { comp = 3; hy = (l - 5) & 1; hz = (l - 5) >> 1; }
    else if (l < 11) { comp = 4; hz = l - 9; }
    else { comp = 5; hy = (l - 11) & 1; }
  }
  off = comp * fvol;
  sgx = sgy = sgz = 0.f;
  if (hx >= 0) { off += hx - 1; sgx = 0.5f - (float)hx; }
  if (hy >= 0) { off += (hy - 1) * fs1; sgy = 0.5f - (float)hy; }
  if (hz >= 0) { off += (hz - 1) * fs2; sgz = 0.5f - (float)hz; }
}

// one lane = one piece: the polynomial coefficients of its component around base point q
// 2-d: f = c0 + ay c1 + az c2 + ay az c3;  3-d: coefficient of ax^i ay^j az^k at [i + 2 j + 4 k]
template <bool D3>
__device__ __forceinline__ void piece_build(float *__restrict__ t, const float *__restrict__ q, int fs1,
                                            int fs2, float sgx, float sgy, float sgz) {
  if (D3) {
    float c[8];
#pragma unroll
    for (int k = 0; k < 2; k++)
#pragma unroll
      for (int j = 0; j < 2; j++) {
        const float v0 = q[k * fs2 + j * fs1], v1 = q[k * fs2 + j * fs1 + 1];
        const float d = v1 - v0;
        c[4 * k + 2 * j] = fmaf(sgx, d, v0);
        c[4 * k + 2 * j + 1] = d;
      }
#pragma unroll
    for (int k = 0; k < 2; k++)
#pragma unroll
      for (int i = 0; i < 2; i++) {
        const float d = c[4 * k + 2 + i] - c[4 * k + i];
        c[4 * k + i] = fmaf(sgy, d, c[4 * k + i]);
        c[4 * k + 2 + i] = d;
      }
#pragma unroll
    for (int i = 0; i < 4; i++) {
      const float d = c[4 + i] - c[i];
      c[i] = fmaf(sgz, d, c[i]);
      c[4 + i] = d;
    }
    reinterpret_cast<float4 *>(t)[0] = make_float4(c[0], c[1], c[2], c[3]);
    reinterpret_cast<float4 *>(t)[1] = make_float4(c[4], c[5], c[6], c[7]);
  } else {
    const float v00 = q[0], v10 = q[1], v01 = q[fs2], v11 = q[fs2 + 1];
    const float d1 = v10 - v00, d2 = v01 - v00, d3 = (v11 - v10) - d2;
    const float c2 = fmaf(sgy, d3, d2);
    *reinterpret_cast<float4 *>(t) = make_float4(fmaf(sgz, c2, fmaf(sgy, d1, v00)), fmaf(sgz, d3, d1), c2, d3);
  }
}

template <bool D3>
__device__ __forceinline__ float piece_eval(const float *__restrict__ t, float ax, float ay, float az) {
  if (D3) {
    const float4 a = reinterpret_cast<const float4 *>(t)[0], b = reinterpret_cast<const float4 *>(t)[1];
    const float lo = fmaf(ay, fmaf(ax, a.w, a.z), fmaf(ax, a.y, a.x));
    const float hi = fmaf(ay, fmaf(ax, b.w, b.z), fmaf(ax, b.y, b.x));
    return fmaf(az, hi, lo);
  } else {
    const float4 a = *reinterpret_cast<const float4 *>(t);
    return fmaf(az, fmaf(ay, a.w, a.z), fmaf(ay, a.y, a.x));
  }
}

// b1 gather of one component (Eq. 11; each component from its own staggered
// points).  q points at the first stencil point, f* are the weights of the second point.
template <bool D3>
__device__ __forceinline__ float gather1(const float *__restrict__ q, int s1, int s2, float fx,
                                         float fy, float fz) {
  if (D3) {
    const float v00 = fmaf(fx, q[1] - q[0], q[0]);
    const float v10 = fmaf(fx, q[s1 + 1] - q[s1], q[s1]);
    const float v01 = fmaf(fx, q[s2 + 1] - q[s2], q[s2]);
    const float v11 = fmaf(fx, q[s2 + s1 + 1] - q[s2 + s1], q[s2 + s1]);
    const float w0 = fmaf(fy, v10 - v00, v00);
    const float w1 = fmaf(fy, v11 - v01, v01);
    return fmaf(fz, w1 - w0, w0);
  } else {
    const float w0 = fmaf(fy, q[1] - q[0], q[0]);
    const float w1 = fmaf(fy, q[s2 + 1] - q[s2], q[s2]);
    return fmaf(fz, w1 - w0, w0);
  }
}

// XC: optional columns may be bound (the carried invariant coordinate of a 2-d run, the id).
// BIG == false: the cells that fit the shared-memory image (store.cuh); BIG == true: a second
// launch for the tiles in which the first one had to leave a cell out.
// TM: the E/B tile arrives by two TMA tensor copies (one box of 8 x 6 x 6 x 3 values per field
// array) and the J tile leaves by one TMA tensor reduction (add) -- three instructions of one
// thread instead of 1300 4-byte copies and 1000 atomics with their index arithmetic.
template <bool D3, int CBS, int THREADS, int MINB, bool XC, bool BIG, int CT, bool ALT, bool TM = false>
__global__ void __launch_bounds__(THREADS, MINB)
k_push1(GridDesc gd, StoreDesc sd, const float *__restrict__ E, const float *__restrict__ B,
        float *__restrict__ J, int wstride, const __grid_constant__ TileMaps tm) {
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
  constexpr int NV = D3 ? 12 : 8;
  using Walker = CellWalker<D3, XC, BIG, CT>;
  static_assert(!TM || (D3 && CBS == 4 && !BIG), "TMA tiles: the 3-d default block, image launch");
  TileGeom<D3, CBS, TM> tg;
  tg.init(gd, tile);
  const int lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
  // (broadcast from lane 0: lets the compiler keep everything derived from the warp index uniform)
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
  // per-warp areas first (128-byte aligned cell images), then the block's tiles and tables
  constexpr int QROWS = D3 ? QROWS3 : QROWS2, QCAP = QCap<D3>::v;
  float *myQ = (float *)(smraw + (size_t)nwarps * wstride) + warp * (QROWS * QCAP);  // [QROWS][QCAP]
  // [NP][W] per warp: the gather table of the warp's current cell (16-byte aligned)
  float *myT = (float *)(smraw + (size_t)nwarps * wstride) + nwarps * (QROWS * QCAP) + warp * GTab<D3>::FLOATS;
  float *sF = (float *)(smraw + (size_t)nwarps * wstride) + nwarps * (QROWS * QCAP + GTab<D3>::FLOATS);  // [6][fvol]
  float *sJ = sF + 6 * tg.fvol;               // [3][jvol]
  uint64_t *tbar = (uint64_t *)(sJ + 3 * tg.jvol);  // TM: mbarrier of the tile loads (8-byte aligned)
  float *sH = sJ + 3 * tg.jvol + (TM ? 2 : 0);  // [8]: Boris h per species
  int *sRel = (int *)(sH + PSC_MAX_SPECIES);  // [24]: J points of vb_values (tile, global)
  int *sNbT = sRel + 24;                      // [27]: first key of the 3^3 neighbouring tiles
  int *sBase = sNbT + 27;                     // [cpb + 1]: first slot of each cell
  int *sCnt = sBase + tg.cpb + 1;             // [cpb]: particles resident in each cell
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
  if (threadIdx.x < 2 * NV) {  // J points of the NV in-cell currents, relative to the cell's node:
    // [0, NV) in the block's J tile, [NV, 2 NV) in the global array
    const bool glob = threadIdx.x >= NV;
    const int i = glob ? threadIdx.x - NV : threadIdx.x;
    const int s1 = glob ? gd.st[1] : tg.je[0], s2 = glob ? gd.st[2] : tg.je[0] * tg.je[1];
    const int jv = glob ? gd.comp : tg.jvol;
    const int off3[12] = {0, s1, s2, s1 + s2, jv, jv + s2, jv + 1, jv + s2 + 1,
                          2 * jv, 2 * jv + 1, 2 * jv + s1, 2 * jv + s1 + 1};
    const int off2[8] = {0, s1, s2, s2 + s1, jv, jv + s2, 2 * jv, 2 * jv + s1};
    sRel[threadIdx.x] = D3 ? off3[i] : off2[i & 7];
  }
  // (asynchronous copies: all of a thread's requests are in flight together)
  for (int i = threadIdx.x; i <= tg.cpb; i += blockDim.x) {
    cp_async4(sBase + i, sd.base + kbase + i, true);
    if (i < tg.cpb) cp_async4(sCnt + i, sd.cnt + kbase + i, true);
  }
  // Without swizzle the box of a TMA tensor copy must start on a 16-byte boundary along x (measured:
  // an x coordinate that is not a multiple of 4 floats raises "illegal instruction"), so the TMA
  // tiles start one point further left (stored x = o, a multiple of 4) and every tile x index is
  // one larger: XS.
  constexpr int XS = TM ? 1 : 0;
  const int tc0 = D3 ? tg.o[0] - 1 - XS + gd.g[0] : 0, tc1 = tg.o[1] - 1 + gd.g[1], tc2 = tg.o[2] - 1 + gd.g[2];
  if (TM) {
    if (threadIdx.x == 0) {
      mbar_init(tbar, 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
      mbar_expect_tx(tbar, 2u * 3u * (unsigned)tg.fvol * 4u);
      tma_load_4d(sF, &tm.E, tc0, tc1, tc2, 0, tbar);
      tma_load_4d(sF + 3 * tg.fvol, &tm.B, tc0, tc1, tc2, 0, tbar);
    }
  } else
  for (int i = threadIdx.x; i < 6 * tg.fvol; i += blockDim.x) {
    const int c = i / tg.fvol, r = i - c * tg.fvol;
    const int lx = r % tg.fe[0], t = r / tg.fe[0];
    const int ly = t % tg.fe[1], lz = t / tg.fe[1];
    const int gx = D3 ? tg.o[0] + lx - 1 + gd.g[0] : 0;
    const int gy = tg.o[1] + ly - 1 + gd.g[1], gz = tg.o[2] + lz - 1 + gd.g[2];
    const int gi = (gz * gd.ext[1] + gy) * gd.ext[0] + gx;
    cp_async4(sF + i, c < 3 ? E + c * gd.comp + gi : B + (c - 3) * gd.comp + gi, true);
  }
  cp_async_commit();
  for (int i = threadIdx.x; i < 3 * tg.jvol; i += blockDim.x) sJ[i] = 0.f;
  cp_async_wait<0>();
  __syncthreads();
  if (TM) mbar_wait(tbar, 0);  // (after the barrier: thread 0's mbarrier.init is visible)

  const int fs1 = tg.fe[0], fs2 = tg.fe[0] * tg.fe[1], fvol = tg.fvol;
  const unsigned lt = lanemask_lt_();
  const float cdx = D3 ? gd.dt_dx[0] : 0.f, cdy = gd.dt_dx[1], cdz = gd.dt_dx[2];

  // (which reduced value a lane ends up holding after the per-cell reduction, and the J point it
  // belongs to, is recomputed per cell: lane constants kept across the particle loop cost registers)
  int qcnt = 0;  // warp-uniform: entries in this warp's queue
  // global index of the node of the tile's first cell
  const int gnode0 = ((tg.o[2] + gd.g[2]) * gd.ext[1] + (tg.o[1] + gd.g[1])) * gd.ext[0] + (D3 ? tg.o[0] + gd.g[0] : 0);

  // One particle: gather (Eq. 11 with b1 weights; each component from its own Yee points:
  // node-centred along d: points l, l+1, weight a; half-staggered: points l-1, l (a < 1/2, weight
  // a + 1/2) or l, l+1 (weight a - 1/2)), Boris (Eq. 27-28).  ALT: the alternating-order scheme
  // (A29): along a half-staggered direction the weight is b0, i.e. the
  // cell's own point l with weight 1.
  // this lane's piece of the gather table (lanes >= NP: none)
  // packed in one register: offset << 6 | twice the three weight shifts as 2-bit signed fields
  int pc_desc;
  {
    int off;
    float sx_, sy_, sz_;
    piece_desc<D3>(lane < GTab<D3>::NP ? lane : 0, fs1, fs2, fvol, off, sx_, sy_, sz_);
    pc_desc = (off << 6) | (((int)(2.f * sx_) & 3) << 4) | (((int)(2.f * sy_) & 3) << 2) | ((int)(2.f * sz_) & 3);
  }
  auto kick = [&](const float *cF, float ax, float ay, float az, float &ux, float &uy, float &uz, int sp) {
    if (!ALT) {  // the cell's gather table (built at the start of the cell)
      constexpr int W = GTab<D3>::W;
      const int iy = ay >= 0.5f ? W : 0, iz = az >= 0.5f ? W : 0, ix = (D3 && ax >= 0.5f) ? W : 0;
      float ex, ey, ez, bx, by, bz;
      if (D3) {
        ex = piece_eval<D3>(myT + ix, ax, ay, az);
        ey = piece_eval<D3>(myT + 2 * W + iy, ax, ay, az);
        ez = piece_eval<D3>(myT + 4 * W + iz, ax, ay, az);
        bx = piece_eval<D3>(myT + 6 * W + iy + 2 * iz, ax, ay, az);
        by = piece_eval<D3>(myT + 10 * W + ix + 2 * iz, ax, ay, az);
        bz = piece_eval<D3>(myT + 14 * W + ix + 2 * iy, ax, ay, az);
      } else {
        ex = piece_eval<D3>(myT, ax, ay, az);
        ey = piece_eval<D3>(myT + W + iy, ax, ay, az);
        ez = piece_eval<D3>(myT + 3 * W + iz, ax, ay, az);
        bx = piece_eval<D3>(myT + 5 * W + iy + 2 * iz, ax, ay, az);
        by = piece_eval<D3>(myT + 9 * W + iz, ax, ay, az);
        bz = piece_eval<D3>(myT + 11 * W + iy, ax, ay, az);
      }
      boris_push(ux, uy, uz, ex, ey, ez, bx, by, bz, sH[sp & (PSC_MAX_SPECIES - 1)]);
      return;
    }
    const bool hy = ALT || ay >= 0.5f, hz = ALT || az >= 0.5f, hx = D3 && (ALT || ax >= 0.5f);
    const float gy = ALT ? 0.f : (hy ? ay - 0.5f : ay + 0.5f), gz = ALT ? 0.f : (hz ? az - 0.5f : az + 0.5f);
    const float gx = ALT ? 0.f : (hx ? ax - 0.5f : ax + 0.5f);
    const int oy = hy ? 0 : -fs1, oz = hz ? 0 : -fs2, ox = (!D3 || hx) ? 0 : -1;
    const float ex = gather1<D3>(cF + ox, fs1, fs2, gx, ay, az);
    const float ey = gather1<D3>(cF + fvol + oy, fs1, fs2, ax, gy, az);
    const float ez = gather1<D3>(cF + 2 * fvol + oz, fs1, fs2, ax, ay, gz);
    const float bx = gather1<D3>(cF + 3 * fvol + oy + oz, fs1, fs2, ax, gy, gz);
    const float by = gather1<D3>(cF + 4 * fvol + ox + oz, fs1, fs2, gx, ay, gz);
    const float bz = gather1<D3>(cF + 5 * fvol + ox + oy, fs1, fs2, gx, gy, az);
    boris_push(ux, uy, uz, ex, ey, ez, bx, by, bz, sH[sp & (PSC_MAX_SPECIES - 1)]);
  };
  // The move x^{n+1/2} -> x^{n+3/2} (Eq. 26) in cells, written with explicit roundings: the pass
  // over a cell's leavers recomputes it from the stored momentum and must get the same bits.
  auto move = [&](float ax, float ay, float az, float ux, float uy, float uz, float &vx, float &endx,
                  float &endy, float &endz) {
    const float ig = rsqrt_ge1(__fmaf_rn(ux, ux, __fmaf_rn(uy, uy, __fmaf_rn(uz, uz, 1.0f))));
    vx = __fmul_rn(ux, ig);
    endx = D3 ? __fmaf_rn(vx, cdx, ax) : 0.f;
    endy = __fmaf_rn(__fmul_rn(uy, ig), cdy, ay);
    endz = __fmaf_rn(__fmul_rn(uz, ig), cdz, az);
  };
  // a trajectory that leaves its cell: its record goes to the cell's exchange row (offsets
  // relative to the destination cell), its current through the queue (all its segments)
  auto depart = [&](bool cross, int xi, int packed, int lx, int ly, int lz, float ax, float ay, float az,
                    float endx, float endy, float endz, float vx, float ux, float uy, float uz, float qw,
                    int sp, float x2d, int id) {
    const unsigned cm = __ballot_sync(0xffffffffu, cross);
    if (qcnt + __popc(cm) > QCAP) {  // no room for this batch: walk (up to 32 of) what is queued first
      const int nd = qcnt < 32 ? qcnt : 32;
      qcnt -= nd;
      drain_queue<D3>(J, tg, gd, gnode0, myQ, sRel + NV, qcnt, nd, lane);
    }
    if (cross) {
      const int sxd = D3 ? (endx >= 1.f ? 1 : (endx < 0.f ? -1 : 0)) : 0;
      const int syd = endy >= 1.f ? 1 : (endy < 0.f ? -1 : 0);
      const int szd = endz >= 1.f ? 1 : (endz < 0.f ? -1 : 0);
      // A non-finite end position (a non-finite momentum: PSC_F_NAN) fails every comparison
      // above and would travel under the code of "no move", which no cell collects.  Such a
      // particle keeps its old offsets and goes through the spill list back into its own cell,
      // so that the population stays complete.
      const bool nowhere = (sxd | syd | szd) == 0;
      Part pr;
      pr.ax = D3 ? fminf(fmaxf(endx - (float)sxd, 0.f), 0.99999994f) : 0.f;
      pr.ay = fminf(fmaxf(endy - (float)syd, 0.f), 0.99999994f);
      pr.az = fminf(fmaxf(endz - (float)szd, 0.f), 0.99999994f);
      if (nowhere) { pr.ax = ax; pr.ay = ay; pr.az = az; }
      pr.ux = ux; pr.uy = uy; pr.uz = uz; pr.qw = qw; pr.sp = sp;
      float w[8];
      Walker::to_words(w, pr, x2d);
      int dest = 0;
      if (xi >= PSC_XCAP || nowhere)
        dest = cell_key(gd, D3 ? wrap_cell(tg.o[0] + lx + sxd, gd.n[0]) : 0,
                        wrap_cell(tg.o[1] + ly + syd, gd.n[1]), wrap_cell(tg.o[2] + lz + szd, gd.n[2]));
      wk.emit(sd, nowhere ? PSC_XCAP : xi, dir_code<D3>(sxd, syd, szd), w, id, dest);
      const int e = qcnt + __popc(cm & lt);
      if (QCAP >= 32 || e < QCAP) {
        myQ[0 * QCAP + e] = __int_as_float(packed);
        if (D3) myQ[1 * QCAP + e] = ax;
        myQ[2 * QCAP + e] = ay;
        myQ[3 * QCAP + e] = az;
        myQ[4 * QCAP + e] = D3 ? endx : vx;
        myQ[5 * QCAP + e] = endy;
        myQ[6 * QCAP + e] = endz;
        myQ[(D3 ? 7 : 1) * QCAP + e] = qw;
      } else {  // a batch of more than QCAP leavers (the BIG form only): the rest is walked at once
        vb_walk<D3, decltype(tg)>(J, gd, gnode0, lx, ly, lz, ax, ay, az, endx, endy, endz, qw * gd.cur[0],
                                  qw * gd.cur[1], qw * gd.cur[2], qw * gd.inv_dV * vx, sRel + NV);
      }
    }
    qcnt += __popc(cm);
    if (QCAP < 32 && qcnt > QCAP) qcnt = QCAP;
    __syncwarp();
    // (a well-filled queue is walked after the cell, while the next cell's run is being fetched)
  };

  // The warp's cells: warp, warp + nwarps, ...  The header words that tell a cell's arrivals are
  // requested one cell ahead; the resident run of the next cell is requested from the copy engine
  // as soon as the image of the current one has been written back.
  int src_next;
  unsigned mask_next = wk.fetch_mask(sd, tg, warp, src_next);
#pragma unroll 1
  for (int ci = warp; ci < tg.cpb; ci += nwarps) {
    const int nx = ci + nwarps;
    const int next_n = nx < tg.cpb ? sCnt[nx] : 0, next_base = nx < tg.cpb ? sBase[nx] : 0;
    const unsigned mask = mask_next;
    const int src = src_next;
    mask_next = wk.fetch_mask(sd, tg, nx, src_next);
    const int lx = ci % tg.bs[0];
    const int lt_ = ci / tg.bs[0];
    const int ly = lt_ % tg.bs[1], lz = lt_ / tg.bs[1];
    // node (lx, ly, lz) of the field tile (tile point t <-> node o + t - 1)
    const float *cF = sF + (D3 ? ((lz + 1) * tg.fe[1] + (ly + 1)) * tg.fe[0] + (lx + 1 + XS)
                               : (lz + 1) * tg.fe[1] + (ly + 1));
    if (!ALT) {  // the cell's gather table, while its resident run is still on its way
      if (lane < GTab<D3>::NP) {
        auto half = [](int two_bits_at_top) { return 0.5f * (float)(two_bits_at_top >> 30); };
        const int pd = keep_in_loop(pc_desc);
        piece_build<D3>(myT + lane * GTab<D3>::W, cF + (pd >> 6), fs1, fs2, half(pd << 26), half(pd << 28),
                        half(pd << 30));
      }
      __syncwarp();
    }
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
    const int ntot = wk.n + wk.na;
    const int packed = lx | (ly << 10) | (lz << 20);
    float acc[NV];
#pragma unroll
    for (int i = 0; i < NV; i++) acc[i] = 0.f;

    if (!BIG) {
      // ---- image path: every particle of the cell, arrivals included, is a slot of the image ----
      if (wk.na) wk.stage_arrivals(sd);
      auto chunk = [&](int v0, bool act) {
        Part p;
        wk.load_image(v0 + lane, p);
        kick(cF, p.ax, p.ay, p.az, p.ux, p.uy, p.uz, p.sp);
        float vx;
        Part pn = p;
        move(p.ax, p.ay, p.az, p.ux, p.uy, p.uz, vx, pn.ax, pn.ay, pn.az);
        const bool stay = (!D3 || (pn.ax >= 0.f && pn.ax < 1.f)) && pn.ay >= 0.f && pn.ay < 1.f &&
                          pn.az >= 0.f && pn.az < 1.f;
        // Villasenor-Buneman: a trajectory that stays in the cell is one segment, summed in registers
        const float qs = stay ? p.qw : 0.f;
        vb_moments<D3>(acc, p.ax, p.ay, p.az, pn.ax, pn.ay, pn.az, qs * gd.cur[0], qs * gd.cur[1],
                       qs * gd.cur[2], qs * gd.inv_dV * vx);
        wk.store_image(v0, act, !stay, pn);
      };
      // the chunks that hold residents only (every lane a particle, nothing to wait for), then the
      // rest: the residents' tail and the arrivals behind it
      if (!D3) {
        int v0 = 0;
#pragma unroll 1
        for (; v0 + 32 <= wk.n; v0 += 32) chunk(v0, true);
        if (v0 < ntot) {
          wk.arrivals_landed();
#pragma unroll 1
          for (; v0 < ntot; v0 += 32) chunk(v0, v0 + lane < ntot);
        }
      } else {  // (3-d: one copy of the larger chunk body; two cost more in instruction fetch than they save)
        bool landed = false;
#pragma unroll 1
        for (int v0 = 0; v0 < ntot; v0 += 32) {
          if (!landed && v0 + 32 > wk.n) {
            wk.arrivals_landed();
            landed = true;
          }
          chunk(v0, v0 + lane < ntot);
        }
      }
      // ---- the cell's leavers, 32 at a time: records + the currents of their trajectories ------
      const int nl = wk.nh;
#pragma unroll 1
      constexpr int LB = QCAP < 32 ? QCAP : 32;  // a batch of leavers fits the empty queue
      for (int i0 = 0; i0 < nl; i0 += LB) {
        const bool al = lane < LB && i0 + lane < nl;
        Part q;
        float qx2d = 0.f;
        int qid = 0;
        q.ax = q.ay = q.az = 0.25f; q.ux = q.uy = q.uz = q.qw = 0.f; q.sp = 0;
        if (al) wk.leaver(sd, i0 + lane, q, qx2d, qid);
        float qvx, qex, qey, qez;
        move(D3 ? q.ax : 0.f, q.ay, q.az, q.ux, q.uy, q.uz, qvx, qex, qey, qez);
        depart(al, i0 + lane, packed, lx, ly, lz, D3 ? q.ax : 0.f, q.ay, q.az, qex, qey, qez, qvx, q.ux,
               q.uy, q.uz, q.qw, q.sp & (PSC_MAX_SPECIES - 1), qx2d, qid);
      }
    } else {
      // ---- global path: residents from the columns, arrivals from the rows, compaction in place
#pragma unroll 1
      for (int v0 = 0; v0 < ntot; v0 += 32) {
        Part cur;
        float x2d;
        int id;
        const bool act = wk.load_global(sd, v0, cur, x2d, id);
        const float ax = D3 ? cur.ax : 0.f, ay = cur.ay, az = cur.az, qw = cur.qw;
        float ux = cur.ux, uy = cur.uy, uz = cur.uz;
        const int sp = cur.sp & (PSC_MAX_SPECIES - 1);
        kick(cF, ax, ay, az, ux, uy, uz, sp);
        float vx, endx, endy, endz;
        move(ax, ay, az, ux, uy, uz, vx, endx, endy, endz);
        const bool stay = (!D3 || (endx >= 0.f && endx < 1.f)) && endy >= 0.f && endy < 1.f &&
                          endz >= 0.f && endz < 1.f;
        const bool cross = act && !stay;
        const float qs = (cross || !act) ? 0.f : qw;
        vb_moments<D3>(acc, ax, ay, az, endx, endy, endz, qs * gd.cur[0], qs * gd.cur[1],
                       qs * gd.cur[2], qs * gd.inv_dV * vx);
        if (__any_sync(0xffffffffu, cross)) {
          const int xi = wk.leaver_slot(cross);
          depart(cross, xi, packed, lx, ly, lz, ax, ay, az, endx, endy, endz, vx, ux, uy, uz, qw, sp, x2d, id);
        }
        Part pn;
        pn.ax = endx; pn.ay = endy; pn.az = endz;
        pn.ux = ux; pn.uy = uy; pn.uz = uz; pn.qw = qw; pn.sp = sp;
        wk.store_global(sd, act && stay, pn, x2d, id);
      }
    }

    // ---- the cell is done.  First its image goes back to global memory and the next cell's run
    // is requested: everything below needs no image and runs while that request is in flight.
    if (BIG) wk.end_global(sd);
    else wk.end_image(sd, next_n, next_base);
    if (qcnt >= (QCAP < 32 ? 16 : 32)) {
      const int nd = qcnt < 32 ? qcnt : 32;
      qcnt -= nd;
      drain_queue<D3>(J, tg, gd, gnode0, myQ, sRel + NV, qcnt, nd, lane);
    }
    // the in-cell currents take one warp reduction and one shared add per J point
    if (ntot) {
      float r;
      moments_to_values<D3>(acc);
      if (D3) r = warp_reduce12(reinterpret_cast<const float(&)[12]>(acc), lane);
      else r = warp_reduce8(reinterpret_cast<const float(&)[8]>(acc), lane);
      if (!(fabsf(r) < 3.0e38f)) atomicOr(sd.flags, PSC_F_NAN);  // a non-finite momentum poisons the cell's sums
      const int ln = keep_in_loop(lane);
      const bool writer = D3 ? ((ln & 1) == 0 && !((ln & 2) && (ln & 4))) : ((ln & 3) == 0);
      if (writer) {
        const int my_off = sRel[D3 ? red12_index(ln) : ((ln >> 2) & 7)];
        const int node = D3 ? ((lz + 1) * tg.je[1] + (ly + 1)) * tg.je[0] + (lx + 1 + XS)
                            : (lz + 1) * tg.je[1] + (ly + 1);
        atomicAdd(&sJ[node + my_off], r);
      }
    }
  }
  if (qcnt) drain_queue<D3>(J, tg, gd, gnode0, myQ, sRel + NV, 0, qcnt, lane);
  wk.finish();
  if (TM) fence_proxy_async();  // this thread's adds to the J tile, for the TMA reduction below
  __syncthreads();
  if (BIG && threadIdx.x == 0) sd.bigflag[tile] = 0;  // taken care of: the flag is the image launch's to set

  // ---- flush the J tile (interior + halo nodes) to global J --------------------------------
  if (TM) {  // one TMA tensor reduction: J[box] += tile (element-wise atomic adds in the L2)
    if (threadIdx.x == 0) {
      tma_reduce_add_4d(&tm.J, sJ, tc0, tc1, tc2, 0);
      bulk_commit();
      bulk_wait_all();
    }
  } else
  for (int i = threadIdx.x; i < 3 * tg.jvol; i += blockDim.x) {
    const float v = sJ[i];
    if (v == 0.f) continue;
    const int c = i / tg.jvol, r = i - c * tg.jvol;
    const int lx = r % tg.je[0], t = r / tg.je[0];
    const int ly = t % tg.je[1], lz = t / tg.je[1];
    const int gx = D3 ? tg.o[0] + lx - 1 + gd.g[0] : 0;
    const int gy = tg.o[1] + ly - 1 + gd.g[1], gz = tg.o[2] + lz - 1 + gd.g[2];
    atomicAdd(&J[c * gd.comp + (gz * gd.ext[1] + gy) * gd.ext[0] + gx], v);
  }
  if (!BIG) break;
  __syncthreads();  // the next tile reuses the shared memory
  }
}

}  // namespace

int psc_push_order1(psc_ctx *c, cudaStream_t s) {
  const GridDesc &gd = c->gd;
  const bool d3 = gd.n[0] > 1 && gd.n[1] > 1 && gd.n[2] > 1;
  const bool d2yz = gd.n[0] == 1 && gd.n[1] > 1 && gd.n[2] > 1;
  if (!d3 && !d2yz) return PSC_ERR_UNSUPPORTED;  // 2-d runs are yz-plane runs
  int fvol = 1, jvol = 1;
  for (int d = 0; d < 3; d++)
    if (gd.n[d] > 1) {
      fvol *= gd.bs[d] + 2;
      jvol *= gd.bs[d] + 3;
    }
  if (gd.bs[0] > 1000 || gd.bs[1] > 1000 || gd.bs[2] > 1000) return PSC_ERR_UNSUPPORTED;
  const StoreDesc sd = psc_store_desc(c);
  const bool xc = sd.icol_id >= 0 || sd.icol_x2d >= 0;
  const size_t tile_bytes = (size_t)(6 * fvol + 3 * jvol + PSC_MAX_SPECIES + 24 + 27 + 2 * gd.cpb + 2) * sizeof(float);
  const size_t qbytes = d3 ? (size_t)QROWS3 * QCap<true>::v * 4 : (size_t)QROWS2 * QCap<false>::v * 4;
  auto stride = [&](int wbytes) { return (wbytes + 127) / 128 * 128; };
  const int ws_img = stride(d3 ? CellWalker<true, true, false>::smem_bytes(sd.imgC, sd.ncol)
                               : CellWalker<false, true, false>::smem_bytes(sd.imgC, sd.ncol));
  const int ws_big = stride(CellWalker<true, true, true>::smem_bytes(sd.imgC, sd.ncol));
  const size_t tbytes = (size_t)(d3 ? GTab<true>::FLOATS : GTab<false>::FLOATS) * 4;  // gather table per warp
  auto smem_of = [&](int threads, int ws) { return (size_t)(threads / 32) * (ws + qbytes + tbytes) + tile_bytes; };
  if (smem_of(128, ws_img) > 200 * 1024) return PSC_ERR_UNSUPPORTED;
  const int big_grid = gd.ntiles < 2 * c->sm_count ? gd.ntiles : 2 * c->sm_count;
  ProfScope ps(c, PSC_PH_PUSH, s);
#define PSC_LAUNCH_PUSH1_(D3_, CBS_, T_, B_, XC_, BIG_, CT_, SMEM_, WS_)                             \
  do {                                                                                             \
    PSC_CUDA_TRY(c, cudaFuncSetAttribute(k_push1<D3_, CBS_, T_, B_, XC_, BIG_, CT_, false>,        \
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(SMEM_))); \
    k_push1<D3_, CBS_, T_, B_, XC_, BIG_, CT_, false><<<(BIG_) ? big_grid : gd.ntiles, T_, SMEM_, s>>>(gd, sd, c->E, c->B, c->J, WS_, c->tmaps); \
    PSC_LAUNCH_CHECK(c);                                                                           \
  } while (0)
  // the alternating-order scheme runs the general instantiation (run-time tile, optional columns)
#define PSC_LAUNCH_PUSH1_ALT(D3_, B_, BIG_, SMEM_, WS_)                                            \
  do {                                                                                             \
    PSC_CUDA_TRY(c, cudaFuncSetAttribute(k_push1<D3_, 0, 128, B_, true, BIG_, 0, true>,            \
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(SMEM_))); \
    k_push1<D3_, 0, 128, B_, true, BIG_, 0, true><<<(BIG_) ? big_grid : gd.ntiles, 128, SMEM_, s>>>(gd, sd, c->E, c->B, c->J, WS_, c->tmaps); \
    PSC_LAUNCH_CHECK(c);                                                                           \
  } while (0)
  // the image launch, then the launch for the cells it had to leave out (its blocks return at
  // once for every other tile).  The library's default tiles without optional columns get the
  // image stride as a compile-time constant.
#define PSC_LAUNCH_PUSH1(D3_, CBS_, T_, B_, FAST_)                                                 \
  do {                                                                                             \
    if (xc) {                                                                                      \
      PSC_LAUNCH_PUSH1_(D3_, CBS_, T_, B_, true, false, 0, smem_of(T_, ws_img), ws_img);           \
      PSC_LAUNCH_PUSH1_(D3_, CBS_, T_, 2, true, true, 0, smem_of(T_, ws_big), ws_big);             \
    } else {                                                                                       \
      if (FAST_ && sd.imgC == 256) PSC_LAUNCH_PUSH1_(D3_, CBS_, T_, B_, false, false, 256, smem_of(T_, ws_img), ws_img); \
      else if (FAST_ && sd.imgC == 192) PSC_LAUNCH_PUSH1_(D3_, CBS_, T_, B_, false, false, 192, smem_of(T_, ws_img), ws_img); \
      else if (FAST_ && sd.imgC == 160) PSC_LAUNCH_PUSH1_(D3_, CBS_, T_, B_, false, false, 160, smem_of(T_, ws_img), ws_img); \
      else if (FAST_ && sd.imgC == 128) PSC_LAUNCH_PUSH1_(D3_, CBS_, T_, B_, false, false, 128, smem_of(T_, ws_img), ws_img); \
      else PSC_LAUNCH_PUSH1_(D3_, CBS_, T_, B_, false, false, 0, smem_of(T_, ws_img), ws_img);     \
      PSC_LAUNCH_PUSH1_(D3_, CBS_, T_, 2, false, true, 0, smem_of(T_, ws_big), ws_big);            \
    }                                                                                              \
  } while (0)
  // 3-d default block, no optional columns, TMA maps available: tiles staged by TMA
  const bool tma3 = d3 && c->have_tmaps && !xc && gd.gmode != PSC_SCHEME_ALTERNATING && gd.bs[0] == 4 &&
                    gd.bs[1] == 4 && gd.bs[2] == 4 && (sd.imgC == 160 || sd.imgC == 128);
  c->used_tma = tma3 ? 1 : 0;
  if (tma3) {
    const size_t tile_tm = (size_t)(6 * 288 + 3 * 392 + 2 + PSC_MAX_SPECIES + 24 + 27 + 2 * gd.cpb + 2) * sizeof(float);
    const size_t smem_tm = (size_t)4 * (ws_img + qbytes + tbytes) + tile_tm;
#define PSC_LAUNCH_PUSH1_TM(CT_)                                                                   \
  do {                                                                                             \
    PSC_CUDA_TRY(c, cudaFuncSetAttribute(k_push1<true, 4, 128, PSC_MINB3D, false, false, CT_, false, true>, \
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_tm)); \
    k_push1<true, 4, 128, PSC_MINB3D, false, false, CT_, false, true><<<gd.ntiles, 128, smem_tm, s>>>( \
        gd, sd, c->E, c->B, c->J, ws_img, c->tmaps);                                               \
    PSC_LAUNCH_CHECK(c);                                                                           \
  } while (0)
    if (sd.imgC == 160) PSC_LAUNCH_PUSH1_TM(160);
    else PSC_LAUNCH_PUSH1_TM(128);
#undef PSC_LAUNCH_PUSH1_TM
    PSC_LAUNCH_PUSH1_(true, 4, 128, 2, false, true, 0, smem_of(128, ws_big), ws_big);  // the BIG launch as usual
  } else if (gd.gmode == PSC_SCHEME_ALTERNATING) {
    if (d3) {
      PSC_LAUNCH_PUSH1_ALT(true, 4, false, smem_of(128, ws_img), ws_img);
      PSC_LAUNCH_PUSH1_ALT(true, 2, true, smem_of(128, ws_big), ws_big);
    } else {
      PSC_LAUNCH_PUSH1_ALT(false, 5, false, smem_of(128, ws_img), ws_img);
      PSC_LAUNCH_PUSH1_ALT(false, 2, true, smem_of(128, ws_big), ws_big);
    }
  } else if (d3) {
    const bool def = gd.bs[0] == 4 && gd.bs[1] == 4 && gd.bs[2] == 4;
    if (def) PSC_LAUNCH_PUSH1(true, 4, 128, PSC_MINB3D, true);
    else PSC_LAUNCH_PUSH1(true, 0, 128, 4, false);
  } else {
    const bool def = gd.bs[1] == 8 && gd.bs[2] == 8;
    if (def) PSC_LAUNCH_PUSH1(false, 8, PSC_THREADS2D, PSC_MINB2D, true);
    else PSC_LAUNCH_PUSH1(false, 0, 128, 5, false);
  }
#undef PSC_LAUNCH_PUSH1
#undef PSC_LAUNCH_PUSH1_
#undef PSC_LAUNCH_PUSH1_ALT
  return PSC_OK;
}


// TMA tensor maps of E, B, J for the 3-d default tiles (psc_bind_fields).  The encoder is a
// driver entry point fetched through the runtime (the library links no libcuda); if it is not
// there, or the layout does not qualify, the kernel stages its tiles with plain copies.
int psc_make_tile_maps(psc_ctx *c) {
  c->have_tmaps = 0;
  const GridDesc &gd = c->gd;
  if (!psc_is3d(gd) || gd.order != 1) return PSC_OK;
  if (gd.bs[0] != 4 || gd.bs[1] != 4 || gd.bs[2] != 4) return PSC_OK;
  if (gd.ext[0] % 4 != 0) return PSC_OK;  // global strides must be multiples of 16 bytes
  typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void *fn = nullptr;
  cudaDriverEntryPointQueryResult qr;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn ||
      qr != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    return PSC_OK;
  }
  const cuuint64_t dims[4] = {(cuuint64_t)gd.ext[0], (cuuint64_t)gd.ext[1], (cuuint64_t)gd.ext[2], 3};
  const cuuint64_t strides[3] = {(cuuint64_t)gd.ext[0] * 4, (cuuint64_t)gd.ext[0] * gd.ext[1] * 4,
                                 (cuuint64_t)gd.comp * 4};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  const cuuint32_t fbox[4] = {8, 6, 6, 3}, jbox[4] = {8, 7, 7, 3};
  struct { CUtensorMap *m; float *p; const cuuint32_t *box; } todo[3] = {
      {&c->tmaps.E, c->E, fbox}, {&c->tmaps.B, c->B, fbox}, {&c->tmaps.J, c->J, jbox}};
  for (auto &t : todo) {
    const CUresult r = ((encode_fn)fn)(t.m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, t.p, dims, strides, t.box, estr,
                                       CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                       CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return PSC_OK;
  }
  c->have_tmaps = 1;
  return PSC_OK;
}
