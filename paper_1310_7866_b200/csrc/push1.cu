// push1.cu -- the fused particle loop of Fig. 8 for first-order
// particles: gather E,B with b1 weights (Eq. 11, 29-31), Boris push (Eq. 27-28),
// move (Eq. 26), Villasenor-Buneman charge-conserving deposit, periodic wrap.
//
// One thread block per sort block ("supercell"): the block stages the E/B values
// its cells can touch (tile + 1 halo point each side) in shared memory and accumulates current
// in a shared J tile (tile + 1 low / 2 high halo nodes) that is flushed to global J once.  A
// warp takes one CELL at a time and walks that cell's slots in chunks of 32, so the cell -- and
// with it every tile address that does not depend on the in-cell offset -- is warp-uniform, the
// gather reads are shared-memory broadcasts, and the currents of the trajectories that stay
// inside the cell (the great majority) are summed in registers over the whole cell and
// reduced across the warp once per cell.
//
// This is the single particle loop of PAPER.md:603 ("only one loop each time step that reads
// and writes all particle data"): a cell's particles are loaded as one contiguous run (the
// stayers of the previous step) plus a short indexed list of arrivals (reorder on load; both
// from the index sort of sort.cu), and the advanced particles are written to the cell's segment
// of the OTHER column set -- those that stay in the cell compacted at the front, the leavers at
// the back with the one-byte direction code of their move; per cell the kernel writes the count
// of each code.  The leavers' codes and the counts are all the next sort reads.
//
// Positions are in the internal form (include/psc.h): in-cell offset a in [0,1) per direction;
// the cell is implied by the segment.  The move is b = a + v dt/dx; a particle that leaves its
// cell (b < 0 or b >= 1; at most one cell per direction) is stored with offset
// b -/+ 1 and the direction code of the move; the index sort turns code + source cell into the
// destination cell with the periodic wrap -- the single-GPU form of the particle exchange
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
#include "push_common.cuh"

namespace {

constexpr int QCAP = 64;   // per-warp queue of trajectories that leave their cell
constexpr int QW = 8;      // words per entry
constexpr int QROWS3 = 12; // rows of the queue in 3-d: the drain reuses drained slots as scratch [NV]
constexpr int NST = 4;        // chunks in the per-warp column ring (NST - 1 in flight)
constexpr int RING_COLS = 9;  // y z ux uy uz qw species [x] [id]


// Tile geometry.  CBS != 0: the sort block is CBS cells along every active direction (the
// library defaults, 8x8 in 2-d and 4x4x4 in 3-d), known at compile time so that every tile
// extent, stride and shared-memory offset folds into an immediate; CBS == 0: run-time block.
template <bool D3, int CBS>
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
    fe[0] = D3 ? bs[0] + 2 : 1;
    fe[1] = bs[1] + 2;
    fe[2] = bs[2] + 2;
    je[0] = D3 ? bs[0] + 3 : 1;
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

// Walks the straight line a -> a + dd (cells; at most one face crossing per direction because
// dt <= dx/2) and deposits every segment -- the slow path of the kernel below,
// taken by the trajectories that leave their cell.
// The segments' currents are added with shared-memory atomics, which are compare-and-swap loops
// for fp32 (ATOMS.CAST.SPIN) and therefore pay for every same-address collision inside the
// warp.  The trajectories drained together come from a few cells and cross the same faces, i.e.
// hit the same J points in the same order; so each lane walks its NV values in a different
// rotation (start = lane mod NV): the values go through a lane-private scratch column `scr`
// ([NV][QCAP], the drained queue slots) and are picked with the rotated index, the point offsets
// from the table `rel` ([NV], the order of vb_values).
template <bool D3, class TG>
__device__ __forceinline__ void vb_walk(float *__restrict__ sJ, const TG &tg, int lx,
                                        int ly, int lz, float ax, float ay, float az, float ddx,
                                        float ddy, float ddz, float fx, float fy, float fz,
                                        float qvx, const int *__restrict__ rel,
                                        float *__restrict__ scr, int rot) {
  constexpr int NV = D3 ? 12 : 8;
  const float endx = ax + ddx, endy = ay + ddy, endz = az + ddz;
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
      const int cx = lx + rx, cy = ly + ry, cz = lz + rz;
      float *node = sJ + (D3 ? ((cz + 1) * tg.je[1] + (cy + 1)) * tg.je[0] + (cx + 1)
                             : (cz + 1) * tg.je[1] + (cy + 1));
#pragma unroll
      for (int i = 0; i < NV; i++) scr[i * QCAP] = v[i];
      int idx = rot;
#pragma unroll
      for (int j = 0; j < NV; j++) {
        atomicAdd(node + rel[idx], scr[idx * QCAP]);
        idx = idx + 1 == NV ? 0 : idx + 1;
      }
    }
    if (which == 3) break;
    if (which == 0) { rx += sxd; tx = 2.f; }
    else if (which == 1) { ry += syd; ty = 2.f; }
    else { rz += szd; tz = 2.f; }
    px = qx; py = qy; pz = qz;
    tprev = t;
  }
}


template <bool D3, class TG>
__device__ __forceinline__ void drain_queue(float *__restrict__ sJ, const TG &tg,
                                            const GridDesc &gd, float *__restrict__ q,
                                            const int *__restrict__ rel, int start, int n, int lane) {
  if (lane < n) {
    const int e = start + lane;
    const int packed = __float_as_int(q[0 * QCAP + e]);
    const float ax = q[1 * QCAP + e], ay = q[2 * QCAP + e], az = q[3 * QCAP + e];
    const float ddx = q[4 * QCAP + e], ddy = q[5 * QCAP + e], ddz = q[6 * QCAP + e];
    const float qw = q[7 * QCAP + e];
    const int lx = packed & 1023, ly = (packed >> 10) & 1023, lz = packed >> 20;
    // 2-d: the x slots carry (unused, v_x): the out-of-plane current needs the velocity
    const float fx = qw * gd.cur[0], fy = qw * gd.cur[1], fz = qw * gd.cur[2];
    const float qvx = D3 ? 0.f : qw * gd.inv_dV * ddx;
    vb_walk<D3>(sJ, tg, lx, ly, lz, D3 ? ax : 0.f, ay, az, D3 ? ddx : 0.f, ddy, ddz, fx, fy, fz,
                qvx, rel, q + e, lane % (D3 ? 12 : 8));
  }
  __syncwarp();
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

// XC: optional columns may be bound (the carried invariant coordinate of a 2-d run, the id)
template <bool D3, int CBS, int THREADS, int MINB, bool XC>
__global__ void __launch_bounds__(THREADS, MINB)
k_push1(GridDesc gd, Cols in, Cols out, PushLists pls, const float *__restrict__ E,
        const float *__restrict__ B, float *__restrict__ J, uint32_t *__restrict__ flags) {
  extern __shared__ float smem[];
  constexpr int NV = D3 ? 12 : 8;
  TileGeom<D3, CBS> tg;
  tg.init(gd, blockIdx.x);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  float *sF = smem;                           // [6][fvol]: Ex Ey Ez Bx By Bz
  float *sJ = smem + 6 * tg.fvol;             // [3][jvol]
  float *sH = sJ + 3 * tg.jvol;               // [8]: Boris h per species
  int *sDir = (int *)(sH + PSC_MAX_SPECIES);  // [warps][32]
  constexpr int QR = D3 ? QROWS3 : QW;        // queue rows (>= NV: drained slots serve as scratch)
  float *sQ = (float *)(sDir + nwarps * 32);  // [warps][QR][QCAP]
  float *myQ = sQ + warp * (QR * QCAP);
  float *myRing = sQ + nwarps * (QR * QCAP) + warp * (NST * RING_COLS * 32);  // [NST][RING_COLS][32]
  int *sRel = (int *)(sQ + nwarps * (QR * QCAP + NST * RING_COLS * 32));  // [12]: J points of vb_values
  int *sIn = sRel + 12;                            // [cpb]: first input slot of each cell's run
  int *sNs = sIn + tg.cpb;                         // [cpb]: length of that run
  int *sA = sNs + tg.cpb;                          // [cpb + 1]: first arrival-list entry
  int *sOut = sA + tg.cpb + 1;                     // [cpb + 1]: output segments
  uint8_t *__restrict__ dcode = pls.dcode;
  int *__restrict__ dircnt = pls.dircnt;
  const int *__restrict__ alist = pls.alist;

  if (threadIdx.x < PSC_MAX_SPECIES) sH[threadIdx.x] = gd.qmh[threadIdx.x];
  if (threadIdx.x < NV) {  // J points of the NV in-cell currents, relative to the cell's node
    const int s1 = tg.je[0], s2 = tg.je[0] * tg.je[1], jv = tg.jvol;
    const int off3[12] = {0, s1, s2, s1 + s2, jv, jv + s2, jv + 1, jv + s2 + 1,
                          2 * jv, 2 * jv + 1, 2 * jv + s1, 2 * jv + s1 + 1};
    const int off2[8] = {0, 1, s2, s2 + 1, jv, jv + s2, 2 * jv, 2 * jv + 1};
    sRel[threadIdx.x] = D3 ? off3[threadIdx.x] : off2[threadIdx.x & 7];
  }
  for (int i = threadIdx.x; i < 6 * tg.fvol; i += blockDim.x) {
    const int c = i / tg.fvol, r = i - c * tg.fvol;
    const int lx = r % tg.fe[0], t = r / tg.fe[0];
    const int ly = t % tg.fe[1], lz = t / tg.fe[1];
    const int gx = D3 ? tg.o[0] + lx - 1 + gd.g[0] : 0;
    const int gy = tg.o[1] + ly - 1 + gd.g[1], gz = tg.o[2] + lz - 1 + gd.g[2];
    const int gi = (gz * gd.ext[1] + gy) * gd.ext[0] + gx;
    sF[i] = c < 3 ? E[c * gd.comp + gi] : B[(c - 3) * gd.comp + gi];
  }
  for (int i = threadIdx.x; i < 3 * tg.jvol; i += blockDim.x) sJ[i] = 0.f;
  const int kbase = blockIdx.x * tg.cpb;
  for (int i = threadIdx.x; i <= tg.cpb; i += blockDim.x) {
    const int o = pls.offs_in[kbase + i];
    if (i < tg.cpb) {
      sIn[i] = o;
      sNs[i] = pls.nstay ? pls.nstay[kbase + i] : pls.offs_in[kbase + i + 1] - o;
    }
    sA[i] = pls.aoffs ? pls.aoffs[kbase + i] : 0;
    sOut[i] = pls.offs_out[kbase + i];
  }
  sDir[warp * 32 + lane] = 0;
  __syncthreads();
  for (int i = threadIdx.x; i < tg.cpb; i += blockDim.x)  // empty cells send nothing anywhere
    if (sOut[i + 1] == sOut[i])
      for (int d = 0; d < (D3 ? 27 : 9); d++) dircnt[d * gd.nkeys + kbase + i] = 0;

  const int fs1 = tg.fe[0], fs2 = tg.fe[0] * tg.fe[1], fvol = tg.fvol;
  uint32_t bad = 0;
  const unsigned lt = lanemask_lt_();
  const float cdx = D3 ? gd.dt_dx[0] : 0.f, cdy = gd.dt_dx[1], cdz = gd.dt_dx[2];

  // which reduced value this lane ends up holding, and the J point (relative to the cell's
  // (lx+1, ly+1, lz+1) tile node) it belongs to
  int my_off;
  bool writer;
  if (D3) {
    my_off = sRel[red12_index(lane)];
    writer = (lane & 1) == 0 && !((lane & 2) && (lane & 4));
  } else {
    my_off = sRel[(lane >> 2) & 7];
    writer = (lane & 3) == 0;
  }
  int qcnt = 0;  // warp-uniform: entries in this warp's queue

  // The warp's work is the sequence of 32-particle chunks of its cells (cells warp, warp +
  // nwarps, ...; empty cells skipped).  Particle v of a cell is slot sIn + v of the input columns
  // if v < sNs (the cell's stayer run), else slot alist[sA + v - sNs] (an arrival: reorder on
  // load).  The loop is software-pipelined: the columns of chunk t+1 are loaded before chunk t is
  // computed, and the list entries of chunk t+2 with them, so that a DRAM round trip is hidden
  // behind one chunk of arithmetic.
  struct It {
    int ci, base, p1;  // cell, first particle of the chunk, particles in the cell
    bool ok;
    int ns, in0;       // the cell's stayer run: length, first input slot (per-cell constants kept
                       // in registers: the load/store path of the SM is the scarce resource)
  };
  auto adv = [&](It &it) {
    it.base += 32;
    while (it.base >= it.p1) {
      it.ci += nwarps;
      if (it.ci >= tg.cpb) {
        it.ok = false;
        return;
      }
      it.base = 0;
      it.p1 = sOut[it.ci + 1] - sOut[it.ci];
      it.ns = sNs[it.ci];
      it.in0 = sIn[it.ci];
    }
  };
  struct Raw {
    float ax, ay, az, ux, uy, uz, qw, cx;
    int sp, id;
  };
  auto load_slot = [&](const It &it) -> int {
    const int v = it.base + lane;
    return (v >= it.ns && v < it.p1) ? ld_stream(alist + (sA[it.ci] + v - it.ns)) : it.in0 + v;
  };
  // Particle columns travel through a per-warp shared-memory ring of NST chunks filled with
  // asynchronous 4-byte copies (cp.async; each lane copies and later reads its own element, so no
  // cross-lane synchronisation is involved): NST - 1 chunks of loads are in flight per warp
  // without holding registers, which is what hides the DRAM latency at 20 warps per SM.
  // Lanes past the end of the cell copy zero bytes, i.e. get zero-filled slots.
  const bool has_x = D3 || (XC && in.x != nullptr), has_id = XC && in.id != nullptr;
  auto issue = [&](const It &it, int p, int stage) {
    const bool v = it.base + lane < it.p1;
    const int q = v ? p : 0;
    float *r = myRing + stage * (RING_COLS * 32) + lane;
    cp_async4(r + 0 * 32, in.y + q, v);
    cp_async4(r + 1 * 32, in.z + q, v);
    cp_async4(r + 2 * 32, in.ux + q, v);
    cp_async4(r + 3 * 32, in.uy + q, v);
    cp_async4(r + 4 * 32, in.uz + q, v);
    cp_async4(r + 5 * 32, in.qw + q, v);
    cp_async4(r + 6 * 32, in.sp + q, v);
    if (has_x) cp_async4(r + 7 * 32, in.x + q, v);
    if (has_id) cp_async4(r + 8 * 32, in.id + q, v);
  };
  auto fetch = [&](Raw &r_, int stage) {
    const float *r = myRing + stage * (RING_COLS * 32) + lane;
    r_.ay = r[0 * 32];
    r_.az = r[1 * 32];
    r_.ux = r[2 * 32];
    r_.uy = r[3 * 32];
    r_.uz = r[4 * 32];
    r_.qw = r[5 * 32];
    r_.sp = __float_as_int(r[6 * 32]);
    r_.ax = r_.cx = 0.f;
    if (has_x) {
      const float t = r[7 * 32];
      if (D3) r_.ax = t; else r_.cx = t;
    }
    r_.id = has_id ? __float_as_int(r[8 * 32]) : 0;
  };

  It a = {warp - nwarps, 0, 0, true, 0, 0};  // the chunk to compute
  adv(a);
  It pr = a;                           // the chunk to issue loads for (NST - 1 ahead)
  int pPr = 0;
  if (pr.ok) pPr = load_slot(pr);
  int stage_p = 0, stage_c = 0;
#pragma unroll 1
  for (int k = 0; k < NST - 1; k++) {
    if (pr.ok) {
      issue(pr, pPr, stage_p);
      adv(pr);
      if (pr.ok) pPr = load_slot(pr);
    }
    cp_async_commit();
    stage_p++;
  }
  int ncross = 0, nst = 0;  // warp-uniform: leavers / stayers of the current cell so far
  int cur_ci = -1, lx = 0, ly = 0, lz = 0, packed = 0;
  int oF = 0, oB = 0;  // the cell's output segment: first slot, last slot
  const float *cF = sF;
  float acc[NV];

  while (a.ok) {
    const It c = a;
    if (pr.ok) {
      issue(pr, pPr, stage_p);
      adv(pr);
      if (pr.ok) pPr = load_slot(pr);  // list entries one more chunk ahead
    }
    cp_async_commit();
    stage_p = stage_p + 1 == NST ? 0 : stage_p + 1;
    cp_async_wait<NST - 1>();
    Raw cur;
    fetch(cur, stage_c);
    stage_c = stage_c + 1 == NST ? 0 : stage_c + 1;
    adv(a);  // a: the next chunk (tells whether this one ends its cell)
    if (c.ci != cur_ci) {  // first chunk of a cell
      cur_ci = c.ci;
      lx = c.ci % tg.bs[0];
      const int lt_ = c.ci / tg.bs[0];
      ly = lt_ % tg.bs[1];
      lz = lt_ / tg.bs[1];
      packed = lx | (ly << 10) | (lz << 20);
      oF = sOut[c.ci];
      oB = sOut[c.ci + 1] - 1;
      // node (lx, ly, lz) of the field tile (tile point t <-> node o + t - 1)
      cF = sF + (D3 ? ((lz + 1) * tg.fe[1] + (ly + 1)) * tg.fe[0] + (lx + 1)
                    : (lz + 1) * tg.fe[1] + (ly + 1));
#pragma unroll
      for (int i = 0; i < NV; i++) acc[i] = 0.f;
    }
    {
      const bool act = c.base + lane < c.p1;
      const float ax = cur.ax, ay = cur.ay, az = cur.az, qw = cur.qw;
      float ux = cur.ux, uy = cur.uy, uz = cur.uz;
      const int sp = cur.sp;

      // ---- gather (Eq. 11 with b1 weights; each component from its own Yee points) --------
      // node-centred along d: points l, l+1, weight a; half-staggered: points l-1, l
      // (a < 1/2, weight a + 1/2) or l, l+1 (weight a - 1/2)
      const bool hy = ay >= 0.5f, hz = az >= 0.5f, hx = D3 && ax >= 0.5f;
      const float gy = hy ? ay - 0.5f : ay + 0.5f, gz = hz ? az - 0.5f : az + 0.5f;
      const float gx = hx ? ax - 0.5f : ax + 0.5f;
      const int oy = hy ? 0 : -fs1, oz = hz ? 0 : -fs2, ox = (!D3 || hx) ? 0 : -1;
      const float ex = gather1<D3>(cF + ox, fs1, fs2, gx, ay, az);
      const float ey = gather1<D3>(cF + fvol + oy, fs1, fs2, ax, gy, az);
      const float ez = gather1<D3>(cF + 2 * fvol + oz, fs1, fs2, ax, ay, gz);
      const float bx = gather1<D3>(cF + 3 * fvol + oy + oz, fs1, fs2, ax, gy, gz);
      const float by = gather1<D3>(cF + 4 * fvol + ox + oz, fs1, fs2, gx, ay, gz);
      const float bz = gather1<D3>(cF + 5 * fvol + ox + oy, fs1, fs2, gx, gy, az);

      // ---- Boris (Eq. 27-28) and move (Eq. 26) ----------------------------------------------
      boris_push(ux, uy, uz, ex, ey, ez, bx, by, bz, sH[sp]);
      const float ig = rsqrt_ge1(fmaf(ux, ux, fmaf(uy, uy, fmaf(uz, uz, 1.0f))));
      const float vx = ux * ig;
      const float ddx = D3 ? vx * cdx : 0.f;  // displacement in cells
      const float ddy = (uy * ig) * cdy, ddz = (uz * ig) * cdz;
      const float endx = ax + ddx, endy = ay + ddy, endz = az + ddz;
      const int sxd = D3 ? (endx >= 1.f ? 1 : (endx < 0.f ? -1 : 0)) : 0;
      const int syd = endy >= 1.f ? 1 : (endy < 0.f ? -1 : 0);
      const int szd = endz >= 1.f ? 1 : (endz < 0.f ? -1 : 0);
      const int dc = dir_code<D3>(sxd, syd, szd);
      const bool cross = act && dc != (D3 ? 13 : 4);

      // ---- Villasenor-Buneman deposit ---------------------------------------------------------
      // a trajectory that stays in the cell is one segment: its currents go to the per-cell
      // register sums; one that leaves goes through the per-warp queue (all its segments)
      {
        const float qs = cross ? 0.f : qw;
        vb_moments<D3>(acc, ax, ay, az, endx, endy, endz, qs * gd.cur[0], qs * gd.cur[1],
                       qs * gd.cur[2], qs * gd.inv_dV * vx);
      }
      const unsigned cm = __ballot_sync(0xffffffffu, cross);
      const unsigned sm = __ballot_sync(0xffffffffu, act && !cross);
      // output slot: stayers fill the cell's segment from the front, leavers from the back
      const int s = cross ? oB - ncross - __popc(cm & lt) : oF + nst + __popc(sm & lt);
      nst += __popc(sm);
      if (cm) {
        if (cross) {
          const int e = qcnt + __popc(cm & lt);
          myQ[0 * QCAP + e] = __int_as_float(packed);
          myQ[1 * QCAP + e] = ax;
          myQ[2 * QCAP + e] = ay;
          myQ[3 * QCAP + e] = az;
          myQ[4 * QCAP + e] = D3 ? ddx : vx;
          myQ[5 * QCAP + e] = ddy;
          myQ[6 * QCAP + e] = ddz;
          myQ[7 * QCAP + e] = qw;
        }
        if (cross) atomicAdd(&sDir[warp * 32 + dc], 1);
        qcnt += __popc(cm);
        ncross += __popc(cm);
        __syncwarp();
        if (qcnt >= 32) {
          qcnt -= 32;
          drain_queue<D3>(sJ, tg, gd, myQ, sRel, qcnt, 32, lane);
        }
      }

      // ---- store slot s of the other column set: new offset, momentum, direction code -----
      if (act) {
        const float by_ = fminf(fmaxf(endy - (float)syd, 0.f), 0.99999994f);
        const float bz_ = fminf(fmaxf(endz - (float)szd, 0.f), 0.99999994f);
        if (D3) {
          const float bx_ = fminf(fmaxf(endx - (float)sxd, 0.f), 0.99999994f);
          st_stream(out.x + s, bx_);
          if (!(bx_ >= 0.f)) bad |= PSC_F_NAN;
        } else if (has_x) {
          st_stream(out.x + s, cur.cx);  // invariant coordinate: carried
        }
        st_stream(out.y + s, by_);
        st_stream(out.z + s, bz_);
        st_stream(out.ux + s, ux);
        st_stream(out.uy + s, uy);
        st_stream(out.uz + s, uz);
        st_stream(out.qw + s, qw);
        st_stream(out.sp + s, sp);
        if (has_id) st_stream(out.id + s, cur.id);
        if (cross) dcode[s] = (uint8_t)dc;
        if (!(by_ >= 0.f) || !(bz_ >= 0.f) || !(fabsf(ux) + fabsf(uy) + fabsf(uz) < 3.0e38f)) bad |= PSC_F_NAN;
      }
    }

    // ---- last chunk of the cell: its in-cell currents take one warp reduction and one shared
    // add per J point; its direction-code counts go to the index sort
    if (!a.ok || a.ci != c.ci) {
      float r;
      moments_to_values<D3>(acc);
      if (D3) r = warp_reduce12(reinterpret_cast<const float(&)[12]>(acc), lane);
      else r = warp_reduce8(reinterpret_cast<const float(&)[8]>(acc), lane);
      if (writer) {
        const int node = D3 ? ((lz + 1) * tg.je[1] + (ly + 1)) * tg.je[0] + (lx + 1)
                            : (lz + 1) * tg.je[1] + (ly + 1);
        atomicAdd(&sJ[node + my_off], r);
      }
      // direction-code counts of the cell: the leavers were counted above, the rest stayed
      {
        constexpr int ND = D3 ? 27 : 9, STAY = D3 ? 13 : 4;
        int *row = sDir + warp * 32;
        if (lane < ND) {
          dircnt[lane * gd.nkeys + kbase + c.ci] = lane == STAY ? nst : row[lane];
          row[lane] = 0;
        }
        ncross = 0;
        nst = 0;
        __syncwarp();
      }
    }
  }
  if (qcnt) drain_queue<D3>(sJ, tg, gd, myQ, sRel, 0, qcnt, lane);
  if (bad) atomicOr(flags, bad);
  __syncthreads();

  // ---- flush the J tile (interior + halo nodes) to global J --------------------------------
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
  const int vthreads = 128;
  const int threads = c->opt_threads > 0 ? (c->opt_threads / 32) * 32 : vthreads;
  if (threads < 32 || threads > vthreads) return PSC_ERR_INVALID_ARG;
  const size_t smem = (size_t)(6 * fvol + 3 * jvol + PSC_MAX_SPECIES + (threads / 32) * (32 + (d3 ? QROWS3 : QW) * QCAP + NST * RING_COLS * 32) + 12 + 4 * gd.cpb + 2) * sizeof(float);
  if (gd.bs[0] > 1000 || gd.bs[1] > 1000 || gd.bs[2] > 1000) return PSC_ERR_UNSUPPORTED;
  if (smem > 200 * 1024) return PSC_ERR_UNSUPPORTED;
  const Cols &in = c->cols[c->cur];
  const Cols &out = c->cols[c->cur ^ 1];
  const PushLists pls = psc_push_lists(c);
  ProfScope ps(c, PSC_PH_PUSH, s);
#define PSC_LAUNCH_PUSH1(D3_, CBS_, T_, B_)                                                        \
  do {                                                                                             \
    if (xc) {                                                                                      \
      PSC_CUDA_TRY(c, cudaFuncSetAttribute(k_push1<D3_, CBS_, T_, B_, true>,                       \
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
      k_push1<D3_, CBS_, T_, B_, true><<<gd.ntiles, threads, smem, s>>>(                           \
          gd, in, out, pls, c->E, c->B, c->J, c->d_flags);                                         \
    } else {                                                                                       \
      PSC_CUDA_TRY(c, cudaFuncSetAttribute(k_push1<D3_, CBS_, T_, B_, false>,                      \
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
      k_push1<D3_, CBS_, T_, B_, false><<<gd.ntiles, threads, smem, s>>>(                          \
          gd, in, out, pls, c->E, c->B, c->J, c->d_flags);                                         \
    }                                                                                              \
  } while (0)
  const bool xc = in.id != nullptr || (!d3 && in.x != nullptr);
  if (d3) {
    const bool def = gd.bs[0] == 4 && gd.bs[1] == 4 && gd.bs[2] == 4 && c->opt_push_variant != 2;
    if (def) PSC_LAUNCH_PUSH1(true, 4, 128, 4);
    else PSC_LAUNCH_PUSH1(true, 0, 128, 4);
  } else {
    const bool def = gd.bs[1] == 8 && gd.bs[2] == 8 && c->opt_push_variant != 2;
    if (def && c->opt_push_variant == 1) PSC_LAUNCH_PUSH1(false, 8, 128, 6);
    else if (def) PSC_LAUNCH_PUSH1(false, 8, 128, 5);
    else PSC_LAUNCH_PUSH1(false, 0, 128, 5);
  }
#undef PSC_LAUNCH_PUSH1
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}
