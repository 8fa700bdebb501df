// sort.cu -- cell-key counting sort of the particle list.
//
// One key orders by block ("supercell") and by cell inside the block at once:
//   key = block_index * cells_per_block + cell_in_block.
// A counting sort is O(N + M).  Two forms:
//
// GENERAL (arbitrary input order; the first sort of a run, from absolute positions):
//   1. k_keys     key per particle from floor(fl32(x * 1/dx)) (k_hist: keys already known), and a
//                 histogram over keys with warp-aggregated atomics;
//   2. scan       exclusive prefix sum of the histogram -> cell offsets (three small kernels);
//   3. k_scatter  slot = cursor[key] + rank, again warp-aggregated; writes the permutation;
//   4. k_segsort  the atomics hand out slots in arbitrary order ACROSS warps, so every key's
//                 segment of `perm` is sorted ascending: a set of distinct input indices in
//                 ascending order IS the stable order, hence the result is the unique stable
//                 counting sort, bit-exact against any stable reference;
//   5. k_reorder  out[s] = in[perm[s]] for every column; positions leave in the internal form.
//
// INDEX (steady state: "a particle moves at most one cell per step", "the
// sort only touches keys/indices", "reorder on load"): the list is the previous sort's output
// advanced by one push.  The push wrote every cell's particles back into a segment of the cell's
// size, the STAYERS (still in the cell: the great majority) compacted at the front and the
// LEAVERS at the back, each leaver with the one-byte direction code of its move (one of 9 / 27
// destination classes), and per cell the count of each code.  So the particles of a cell of the
// NEXT step are one contiguous run (its stayers) plus a short list of arrivals, and the sort
// works on cells and leavers only:
//   1. k_dest_hist  per cell: stayers, arrivals (sum over the 8 / 26 neighbour source cells of
//                   the count of the code that points here);
//   2. scan         one pass over (total, arrivals) packed in 64 bits -> new cell offsets and
//                   offsets into the arrival list;
//   3. k_dir_base   first arrival-list slot of every (source cell, code) group: a cell's
//                   arrivals are grouped by the direction they came from;
//   4. k_rank       one warp per source cell walks its LEAVER region and writes the slots of
//                   the leavers into the arrival list.
// No particle column is touched and nothing per stayer is read or written: the next push loads
// the stayer run directly and the arrivals through the list (reorder on load).  The order this
// gives inside a cell (stayers, then arrivals) is a valid cell sort but not the stable one
// (A17); psc_particles_sort, whose contract is the physically sorted, stable list,
// runs the general form on the keys of the written list instead.
#include <limits.h>

#include "psc_internal.cuh"

namespace {

constexpr int SORT_THREADS = 256;
constexpr int SCAN_ITEMS = 8;                         // per thread
constexpr int SCAN_TILE = SORT_THREADS * SCAN_ITEMS;  // 2048 keys per block
constexpr int WARP_SEG_CAP = 1024;                    // ints of shared memory per warp in k_segsort
constexpr int BIG_SMEM_CAP = 48 * 1024;               // ints; larger segments are sorted in global

__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

__global__ void __launch_bounds__(SORT_THREADS)
k_keys(GridDesc gd, int n, const float *__restrict__ x, const float *__restrict__ y,
       const float *__restrict__ z, int *__restrict__ key, int *__restrict__ hist,
       uint32_t *__restrict__ flags) {
  const int a0 = blockIdx.x * blockDim.x + threadIdx.x;
  const int stride = gridDim.x * blockDim.x;
  const int nround = ((n + 31) / 32) * 32;
  for (int a = a0; a < nround; a += stride) {
    const bool valid = a < n;
    int k = -1 - (int)(threadIdx.x & 31);  // distinct per lane: no grouping of invalid lanes
    if (valid) {
      int c[3];
      const float *pos[3] = {x, y, z};
      bool oob = false;
#pragma unroll
      for (int d = 0; d < 3; d++) {
        if (gd.n[d] == 1) {
          c[d] = 0;
          continue;
        }
        const float xi = __fmul_rn(pos[d][a], gd.inv_dx[d]);  // one fp32 rounding, then floor
        int ci = (int)floorf(xi);
        if (!(ci >= 0 && ci < gd.n[d])) {  // also catches NaN
          oob = true;
          ci = ci < 0 ? 0 : gd.n[d] - 1;
          if (xi != xi) ci = 0;
        }
        c[d] = ci;
      }
      if (oob) atomicOr(flags, PSC_F_OOB);
      const int b0 = c[0] / gd.bs[0], b1 = c[1] / gd.bs[1], b2 = c[2] / gd.bs[2];
      const int l0 = c[0] - b0 * gd.bs[0], l1 = c[1] - b1 * gd.bs[1], l2 = c[2] - b2 * gd.bs[2];
      k = ((b2 * gd.nb[1] + b1) * gd.nb[0] + b0) * gd.cpb + (l2 * gd.bs[1] + l1) * gd.bs[0] + l0;
      key[a] = k;
    }
    const unsigned grp = __match_any_sync(0xffffffffu, k);
    if (valid && (grp & lanemask_lt()) == 0) atomicAdd(&hist[k], __popc(grp));
  }
}

// histogram of keys that already exist (internal form: the push wrote them)
__global__ void __launch_bounds__(SORT_THREADS)
k_hist(int n, int nkeys, const int *__restrict__ key, int *__restrict__ hist,
       uint32_t *__restrict__ flags) {
  const int a0 = blockIdx.x * blockDim.x + threadIdx.x;
  const int stride = gridDim.x * blockDim.x;
  const int nround = ((n + 31) / 32) * 32;
  for (int a = a0; a < nround; a += stride) {
    const bool valid = a < n;
    int k = -1 - (int)(threadIdx.x & 31);
    if (valid) {
      k = key[a];
      if (k < 0 || k >= nkeys) {  // cannot happen unless the caller scribbled over the workspace
        atomicOr(flags, PSC_F_OOB);
        k = 0;
      }
    }
    const unsigned grp = __match_any_sync(0xffffffffu, k);
    if (valid && (grp & lanemask_lt()) == 0) atomicAdd(&hist[k], __popc(grp));
  }
}

// key -> cell coordinates
__device__ __forceinline__ void key_to_cell(const GridDesc &gd, int k, int c[3]) {
  const int b = k / gd.cpb, l = k - b * gd.cpb;
  const int b0 = b % gd.nb[0], br = b / gd.nb[0];
  const int b1 = br % gd.nb[1], b2 = br / gd.nb[1];
  const int l0 = l % gd.bs[0], lr = l / gd.bs[0];
  const int l1 = lr % gd.bs[1], l2 = lr / gd.bs[1];
  c[0] = b0 * gd.bs[0] + l0;
  c[1] = b1 * gd.bs[1] + l1;
  c[2] = b2 * gd.bs[2] + l2;
}

__global__ void __launch_bounds__(SORT_THREADS)
k_cell_idx(GridDesc gd, int n, const int *__restrict__ key, int *__restrict__ cell_idx) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n) return;
  int c[3];
  key_to_cell(gd, key[a], c);
  cell_idx[a] = (c[2] * gd.n[1] + c[1]) * gd.n[0] + c[0];
}

// internal form -> absolute positions, in place: x = (cell + offset) * dx
__global__ void __launch_bounds__(SORT_THREADS)
k_to_abs(GridDesc gd, int n, const int *__restrict__ key, float *__restrict__ x,
         float *__restrict__ y, float *__restrict__ z) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n) return;
  int c[3];
  key_to_cell(gd, key[a], c);
  float *pos[3] = {x, y, z};
#pragma unroll
  for (int d = 0; d < 3; d++) {
    if (gd.n[d] == 1) continue;
    // formed in fp64 and rounded once (this pass runs once per export, not per step)
    float v = __double2float_rn(((double)c[d] + (double)pos[d][a]) * (double)gd.dx[d]);
    if (v >= gd.L[d]) v = nextafterf(gd.L[d], 0.f);  // rounding must not leave [0, L)
    pos[d][a] = v;
  }
}

// ---- exclusive scan of in[0..m) -> out[0..m], out[m] = total -----------------------------------
// T = int: one histogram (general sort; cursor := out as well).  T = long long: two histograms
// packed as (hi << 32) | lo and scanned in one pass (index sort: hi = particles per cell, lo =
// arrivals per cell; both totals are < 2^31, so the low half never carries into the high half);
// the last kernel unpacks them into out (hi) and out_lo.

template <typename T>
__device__ __forceinline__ T warp_inclusive(T v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const T t = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += t;
  }
  return v;
}

template <typename T>
__global__ void __launch_bounds__(SORT_THREADS)
k_scan_local(int m, const T *__restrict__ in, T *__restrict__ out, T *__restrict__ tmp) {
  __shared__ T wsum[SORT_THREADS / 32];
  const int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  T v[SCAN_ITEMS];
  T s = 0;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++) {
    v[i] = (base + i < m) ? in[base + i] : (T)0;
    s += v[i];
  }
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const T inc = warp_inclusive(s, lane);
  if (lane == 31) wsum[w] = inc;
  __syncthreads();
  if (w == 0) {
    T t = lane < SORT_THREADS / 32 ? wsum[lane] : (T)0;
    t = warp_inclusive(t, lane);
    if (lane < SORT_THREADS / 32) wsum[lane] = t;
  }
  __syncthreads();
  T run = inc - s + (w ? wsum[w - 1] : (T)0);
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++) {
    if (base + i < m) out[base + i] = run;
    run += v[i];
  }
  if (threadIdx.x == SORT_THREADS - 1) tmp[blockIdx.x] = run;
}

// single block: exclusive scan of tmp[0..nb) in place, tmp[nb] = total
template <typename T>
__global__ void __launch_bounds__(1024) k_scan_tmp(int nb, T *__restrict__ tmp) {
  __shared__ T wsum[32];
  __shared__ T carry_s;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int base = 0; base < nb; base += 1024) {
    const int i = base + threadIdx.x;
    const T v = i < nb ? tmp[i] : (T)0;
    const T inc = warp_inclusive(v, lane);
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    if (w == 0) wsum[lane] = warp_inclusive(wsum[lane], lane);
    __syncthreads();
    const T carry = carry_s;
    const T exc = carry + inc - v + (w ? wsum[w - 1] : (T)0);
    if (i < nb) tmp[i] = exc;
    __syncthreads();
    if (threadIdx.x == 1023) carry_s = exc + v;
    __syncthreads();
  }
  if (threadIdx.x == 0) tmp[nb] = carry_s;
}

__global__ void __launch_bounds__(SORT_THREADS)
k_scan_add(int m, int *__restrict__ out, int *__restrict__ cursor, const int *__restrict__ tmp,
           int nb) {
  const int add = tmp[blockIdx.x];
  const int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++)
    if (base + i < m) {
      const int v = out[base + i] + add;
      out[base + i] = v;
      cursor[base + i] = v;
    }
  if (blockIdx.x == 0 && threadIdx.x == 0) out[m] = tmp[nb];
}

// packed form: loc[] holds the block-local packed scan; out := high halves, out_lo := low halves
__global__ void __launch_bounds__(SORT_THREADS)
k_scan_add2(int m, const long long *__restrict__ loc, int *__restrict__ out,
            int *__restrict__ out_lo, const long long *__restrict__ tmp, int nb) {
  const long long add = tmp[blockIdx.x];
  const int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++)
    if (base + i < m) {
      const long long v = loc[base + i] + add;
      out[base + i] = (int)(v >> 32);
      out_lo[base + i] = (int)(v & 0xffffffffLL);
    }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    out[m] = (int)(tmp[nb] >> 32);
    out_lo[m] = (int)(tmp[nb] & 0xffffffffLL);
  }
}

__global__ void __launch_bounds__(SORT_THREADS)
k_scatter(int n, const int *__restrict__ key, int *__restrict__ cursor, int *__restrict__ perm) {
  const int a0 = blockIdx.x * blockDim.x + threadIdx.x;
  const int stride = gridDim.x * blockDim.x;
  const int nround = ((n + 31) / 32) * 32;
  const int lane = threadIdx.x & 31;
  for (int a = a0; a < nround; a += stride) {
    const bool valid = a < n;
    const int k = valid ? key[a] : -1 - lane;
    const unsigned grp = __match_any_sync(0xffffffffu, k);
    const int leader = __ffs(grp) - 1;
    int base = 0;
    if (valid && lane == leader) base = atomicAdd(&cursor[k], __popc(grp));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (valid) perm[base + __popc(grp & lanemask_lt())] = a;
  }
}

// ---- ascending sort of every key's segment of perm ------------------------------------------

// All-ascending bitonic network ("mirror" first sub-stage): with it, virtual +inf padding past
// n never moves, so pairs whose upper index is >= n are simply skipped.
template <typename Sync>
__device__ __forceinline__ void bitonic_any(int *a, int n, int tid, int nthreads, Sync sync) {
  int P = 1;
  while (P < n) P <<= 1;
  for (int k = 2; k <= P; k <<= 1) {
    const int hk = k >> 1;
    for (int i = tid; i < (P >> 1); i += nthreads) {
      const int blk = i / hk, w = i - blk * hk;
      const int lo = blk * k + w, hi = blk * k + k - 1 - w;
      if (hi < n) {
        const int u = a[lo], v = a[hi];
        if (u > v) {
          a[lo] = v;
          a[hi] = u;
        }
      }
    }
    sync();
    for (int j = hk >> 1; j >= 1; j >>= 1) {
      for (int i = tid; i < (P >> 1); i += nthreads) {
        const int lo = 2 * j * (i / j) + (i % j), hi = lo + j;
        if (hi < n) {
          const int u = a[lo], v = a[hi];
          if (u > v) {
            a[lo] = v;
            a[hi] = u;
          }
        }
      }
      sync();
    }
  }
}

__global__ void __launch_bounds__(SORT_THREADS)
k_segsort(int nkeys, const int *__restrict__ offs, int *__restrict__ perm,
          int *__restrict__ big_list, uint32_t *__restrict__ big_count) {
  __shared__ int buf[SORT_THREADS / 32][WARP_SEG_CAP];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int warps = gridDim.x * (SORT_THREADS / 32);
  for (int k = blockIdx.x * (SORT_THREADS / 32) + w; k < nkeys; k += warps) {
    const int lo = offs[k], n = offs[k + 1] - lo;
    if (n <= 1) continue;
    if (n <= 32) {
      int v = lane < n ? perm[lo + lane] : INT_MAX;
      // already ascending?
      const int nx = __shfl_down_sync(0xffffffffu, v, 1);
      if (__ballot_sync(0xffffffffu, lane < 31 && v > nx) == 0) continue;
#pragma unroll
      for (int kk = 2; kk <= 32; kk <<= 1) {
        {  // mirror sub-stage: partner = mirror image inside the block of kk lanes
          const int p = __shfl_xor_sync(0xffffffffu, v, kk - 1);
          v = (lane ^ (kk - 1)) > lane ? min(v, p) : max(v, p);
        }
#pragma unroll
        for (int j = kk >> 2; j >= 1; j >>= 1) {
          const int p = __shfl_xor_sync(0xffffffffu, v, j);
          v = (lane & j) == 0 ? min(v, p) : max(v, p);
        }
      }
      if (lane < n) perm[lo + lane] = v;
      continue;
    }
    if (n > WARP_SEG_CAP) {
      if (lane == 0) big_list[atomicAdd(big_count, 1u)] = k;
      continue;
    }
    int *b = buf[w];
    bool sorted = true;
    for (int i = lane; i < n; i += 32) b[i] = perm[lo + i];
    __syncwarp();
    for (int i = lane; i < n - 1; i += 32) sorted = sorted && (b[i] <= b[i + 1]);
    if (__all_sync(0xffffffffu, sorted)) continue;
    bitonic_any(b, n, lane, 32, [] { __syncwarp(); });
    for (int i = lane; i < n; i += 32) perm[lo + i] = b[i];
    __syncwarp();
  }
}

// segments longer than WARP_SEG_CAP: one block each (shared memory if it fits, else in place in
// global memory -- slow, only for pathological densities)
__global__ void __launch_bounds__(1024)
k_segsort_big(const int *__restrict__ offs, int *__restrict__ perm,
              const int *__restrict__ big_list, const uint32_t *__restrict__ big_count) {
  extern __shared__ int sbuf[];
  const int nbig = (int)*big_count;
  for (int e = blockIdx.x; e < nbig; e += gridDim.x) {
    const int k = big_list[e];
    const int lo = offs[k], n = offs[k + 1] - lo;
    if (n <= BIG_SMEM_CAP) {
      for (int i = threadIdx.x; i < n; i += blockDim.x) sbuf[i] = perm[lo + i];
      __syncthreads();
      bitonic_any(sbuf, n, threadIdx.x, blockDim.x, [] { __syncthreads(); });
      for (int i = threadIdx.x; i < n; i += blockDim.x) perm[lo + i] = sbuf[i];
      __syncthreads();
    } else {
      bitonic_any(perm + lo, n, threadIdx.x, blockDim.x, [] { __syncthreads(); });
    }
  }
}

// FROM_ABS: the input columns hold absolute positions -> write in-cell offsets
template <bool FROM_ABS>
__global__ void __launch_bounds__(SORT_THREADS)
k_reorder(GridDesc gd, int n, const int *__restrict__ perm, Cols in, Cols out) {
  const int s0 = blockIdx.x * blockDim.x + threadIdx.x;
  const int stride = gridDim.x * blockDim.x;
  for (int s = s0; s < n; s += stride) {
    const int p = perm[s];
    float x = in.x ? in.x[p] : 0.f, y = in.y[p], z = in.z[p];
    const float ux = in.ux[p], uy = in.uy[p], uz = in.uz[p];
    const float qw = in.qw[p];
    const int sp = in.sp[p];
    int id = 0;
    if (in.id) id = in.id[p];
    if (FROM_ABS) {
      // the cell is decided as in k_keys (fp32 product with 1/dx, floor); the offset is then
      // (x - cell dx) / dx with the difference formed by one FMA, i.e. accurate to fp32 RELATIVE
      // precision of the offset also when dx is not a power of two (x * (1/dx) - cell would carry
      // the absolute rounding error of x / dx, ~1e-6 cells at x / dx ~ 20)
      auto rel = [&](float v, int d) {
        const float c = floorf(__fmul_rn(v, gd.inv_dx[d]));
        return fminf(fmaxf(fmaf(-c, gd.dx[d], v) * gd.inv_dx[d], 0.f), 0.99999994f);
      };
      if (gd.n[0] > 1) x = rel(x, 0);
      if (gd.n[1] > 1) y = rel(y, 1);
      if (gd.n[2] > 1) z = rel(z, 2);
    }
    if (in.x) out.x[s] = x;
    out.y[s] = y;
    out.z[s] = z;
    out.ux[s] = ux;
    out.uy[s] = uy;
    out.uz[s] = uz;
    out.qw[s] = qw;
    out.sp[s] = sp;
    if (in.id) out.id[s] = id;
  }
}


// ---- index sort of a pushed list -------------------------------------------------------------

__device__ __forceinline__ int cell_to_key(const GridDesc &gd, const int c[3]) {
  const int b0 = c[0] / gd.bs[0], b1 = c[1] / gd.bs[1], b2 = c[2] / gd.bs[2];
  const int l0 = c[0] - b0 * gd.bs[0], l1 = c[1] - b1 * gd.bs[1], l2 = c[2] - b2 * gd.bs[2];
  return ((b2 * gd.nb[1] + b1) * gd.nb[0] + b0) * gd.cpb + (l2 * gd.bs[1] + l1) * gd.bs[0] + l0;
}

__device__ __forceinline__ int wrap(int c, int n) { return c < 0 ? c + n : (c >= n ? c - n : c); }

// Keys of the 9 / 27 neighbours of a cell without a division per neighbour: the key is a sum of
// one term per direction, key = sum_d (b_d * bstride_d * cpb + l_d * lstride_d), so three
// candidate terms per direction (cell - 1, cell, cell + 1, periodic) give every neighbour by
// three additions.
struct NbKeys {
  int t[3][3];
  __device__ __forceinline__ void init(const GridDesc &gd, const int c[3]) {
    int bstride = gd.cpb, lstride = 1;
#pragma unroll
    for (int d = 0; d < 3; d++) {
#pragma unroll
      for (int s = -1; s <= 1; s++) {
        const int q = wrap(c[d] + s, gd.n[d]);
        const int b = q / gd.bs[d];
        t[d][s + 1] = b * bstride + (q - b * gd.bs[d]) * lstride;
      }
      bstride *= gd.nb[d];
      lstride *= gd.bs[d];
    }
  }
  // neighbour in direction code dc (sign = +1) or the cell that reaches this one by dc (-1)
  template <bool D3>
  __device__ __forceinline__ int key(int dc, int sign) const {
    const int s0 = D3 ? dc % 3 - 1 : 0;
    const int s1 = D3 ? (dc / 3) % 3 - 1 : dc % 3 - 1;
    const int s2 = D3 ? dc / 9 - 1 : dc / 3 - 1;
    return t[0][sign * s0 + 1] + t[1][sign * s1 + 1] + t[2][sign * s2 + 1];
  }
};

// per destination cell k: stayers (its own STAY count), arrivals (source cell k - dir sends
// count[dir]); pack[k] = (stayers + arrivals) << 32 | arrivals for the packed scan
template <bool D3>
__global__ void __launch_bounds__(SORT_THREADS)
k_dest_hist(GridDesc gd, const int *__restrict__ dircnt, int *__restrict__ nstay,
            long long *__restrict__ pack) {
  constexpr int ND = D3 ? 27 : 9, STAY = D3 ? 13 : 4;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= gd.nkeys) return;
  int c[3];
  key_to_cell(gd, k, c);
  NbKeys nb;
  nb.init(gd, c);
  int na = 0;
#pragma unroll
  for (int dc = 0; dc < ND; dc++)
    if (dc != STAY) na += dircnt[dc * gd.nkeys + nb.key<D3>(dc, -1)];
  const int ns = dircnt[STAY * gd.nkeys + k];
  nstay[k] = ns;
  pack[k] = ((long long)(ns + na) << 32) | (long long)na;
}

// dircnt[dc][src] (count, dc != STAY) -> first arrival-list slot of the (src, dc) group, in
// place: the arrivals of a cell are ordered by the direction they came from
template <bool D3>
__global__ void __launch_bounds__(SORT_THREADS)
k_dir_base(GridDesc gd, int *__restrict__ dircnt, const int *__restrict__ aoffs) {
  constexpr int ND = D3 ? 27 : 9, STAY = D3 ? 13 : 4;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= gd.nkeys) return;
  int o = aoffs[k];
  if (aoffs[k + 1] == o) return;  // no arrivals: every group is empty, its base unused
  int c[3];
  key_to_cell(gd, k, c);
  NbKeys nb;
  nb.init(gd, c);
  int cnt[ND];  // all loads first: the stores below may alias them as far as the compiler knows
#pragma unroll
  for (int dc = 0; dc < ND; dc++) cnt[dc] = dc == STAY ? 0 : dircnt[dc * gd.nkeys + nb.key<D3>(dc, -1)];
#pragma unroll
  for (int dc = 0; dc < ND; dc++) {
    if (dc == STAY) continue;
    dircnt[dc * gd.nkeys + nb.key<D3>(dc, -1)] = o;
    o += cnt[dc];
  }
}

// A warp per source cell walks the cell's leaver region of the written list (behind its
// stayers) and writes each leaver's slot into its group of the arrival list.  A region is a
// handful of entries and every step is a dependent global load, so a warp works on RANK_U cells
// at once: their table rows, then their first code chunks, are loaded back to back.
constexpr int RANK_U = 4;

template <bool D3>
__global__ void __launch_bounds__(SORT_THREADS)
k_rank(int nkeys, const int *__restrict__ offs_w, const uint8_t *__restrict__ dcode,
       const int *__restrict__ dirbase, int *__restrict__ alist, uint32_t *__restrict__ flags) {
  constexpr int ND = D3 ? 27 : 9, STAY = D3 ? 13 : 4;
  __shared__ int sb[SORT_THREADS / 32][RANK_U][32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int warps = gridDim.x * (SORT_THREADS / 32);
  const unsigned lt = lanemask_lt();
  for (int k0 = (blockIdx.x * (SORT_THREADS / 32) + w) * RANK_U; k0 < nkeys; k0 += warps * RANK_U) {
    int p0[RANK_U], p1[RANK_U], dc0[RANK_U];
#pragma unroll
    for (int j = 0; j < RANK_U; j++) {
      const int k = k0 + j;
      const bool ok = k < nkeys;
      const int b = (ok && lane < ND) ? dirbase[lane * nkeys + k] : 0;
      sb[w][j][lane] = b;
      p0[j] = (ok ? offs_w[k] : 0) + __shfl_sync(0xffffffffu, b, STAY);
      p1[j] = ok ? offs_w[k + 1] : 0;
    }
#pragma unroll
    for (int j = 0; j < RANK_U; j++) dc0[j] = p0[j] + lane < p1[j] ? (int)dcode[p0[j] + lane] : STAY;
    __syncwarp();
#pragma unroll
    for (int j = 0; j < RANK_U; j++) {
      for (int base = p0[j]; base < p1[j]; base += 32) {
        const int s = base + lane;
        bool act = s < p1[j];
        int dc = base == p0[j] ? dc0[j] : (act ? (int)dcode[s] : STAY);
        if (act && (dc >= ND || dc == STAY)) {  // cannot happen unless the workspace was scribbled over
          atomicOr(flags, PSC_F_OOB);
          act = false;
        }
        // rank inside the (cell, code) group: one ballot per distinct code present (a few);
        // match.any would do it in one instruction but is an order of magnitude slower here
        int rank = 0, cnt = 0;
        unsigned rem = __ballot_sync(0xffffffffu, act);
        while (rem) {
          const int d = __shfl_sync(0xffffffffu, dc, __ffs(rem) - 1);
          const unsigned m = __ballot_sync(0xffffffffu, act && dc == d);
          if (act && dc == d) {
            rank = __popc(m & lt);
            cnt = __popc(m);
          }
          rem &= ~m;
        }
        int slot = 0;
        if (act) slot = sb[w][j][dc] + rank;
        __syncwarp();
        if (act && rank == 0) sb[w][j][dc] += cnt;
        __syncwarp();
        if (act) alist[slot] = s;
      }
    }
    __syncwarp();
  }
}

// key of the particle in slot s of a list laid out by `offs`: the slot's cell, moved by the
// particle's direction code if the slot lies in the cell's leaver region (behind the
// dirtab[cell][STAY] stayers; dirtab == nullptr: a sorted list, nobody has moved)
template <bool D3>
__global__ void __launch_bounds__(SORT_THREADS)
k_slot_keys(GridDesc gd, int n, const int *__restrict__ offs, const int *__restrict__ dirtab,
            const uint8_t *__restrict__ dcode, int *__restrict__ key) {
  constexpr int ND = D3 ? 27 : 9, STAY = D3 ? 13 : 4;
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  int lo = 0, hi = gd.nkeys;  // largest k with offs[k] <= s (and offs[k+1] > s)
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (offs[mid] <= s) lo = mid; else hi = mid;
  }
  int k = lo;
  if (dirtab && s >= offs[k] + dirtab[STAY * gd.nkeys + k]) {
    int c[3];
    key_to_cell(gd, k, c);
    int dc = (int)dcode[s];
    if (dc >= ND) dc = STAY;
    NbKeys nb;
    nb.init(gd, c);
    k = nb.key<D3>(dc, +1);
  }
  key[s] = k;
}

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace

size_t psc_sort_workspace_bytes(const psc_ctx *c, int64_t n) {
  const size_t nk = (size_t)c->gd.nkeys;
  size_t b = 0;
  b += 5 * align_up((size_t)n * 4, 256);                      // key, curkey, perm, cell_idx, alist
  b += align_up((size_t)n, 256);                              // dcode
  b += 5 * align_up((nk + 1) * 4, 256);                       // offs[2], cursor, aoffs, nstay
  b += 2 * align_up((nk + 1) * 8, 256);                       // pack, packloc
  b += align_up(nk * 27 * 4, 256);                            // dircnt
  b += align_up((nk / SCAN_TILE + 3) * 8, 256);               // scan_tmp
  b += align_up(((size_t)n / WARP_SEG_CAP + 16) * 4, 256);    // big_list
  return b;
}

int psc_sort_carve(psc_ctx *c, int64_t n) {
  const size_t nk = (size_t)c->gd.nkeys;
  char *p = (char *)c->ws;
  auto take = [&](size_t bytes) {
    void *r = p;
    p += align_up(bytes, 256);
    return r;
  };
  c->key = (int32_t *)take((size_t)n * 4);
  c->curkey = (int32_t *)take((size_t)n * 4);
  c->perm = (int32_t *)take((size_t)n * 4);
  c->cell_idx = (int32_t *)take((size_t)n * 4);
  c->alist = (int32_t *)take((size_t)n * 4);
  c->dcode = (uint8_t *)take((size_t)n);
  c->offs[0] = (int32_t *)take((nk + 1) * 4);
  c->offs[1] = (int32_t *)take((nk + 1) * 4);
  c->cursor = (int32_t *)take((nk + 1) * 4);
  c->aoffs = (int32_t *)take((nk + 1) * 4);
  c->nstay = (int32_t *)take((nk + 1) * 4);
  c->pack = (long long *)take((nk + 1) * 8);
  c->packloc = (long long *)take((nk + 1) * 8);
  c->dircnt = (int32_t *)take(nk * 27 * 4);
  c->scan_tmp = (long long *)take((nk / SCAN_TILE + 3) * 8);
  c->big_list = (int32_t *)take(((size_t)n / WARP_SEG_CAP + 16) * 4);
  if ((size_t)(p - (char *)c->ws) > c->ws_bytes) return PSC_ERR_WORKSPACE;
  return PSC_OK;
}

namespace {

inline bool is3d(const GridDesc &gd) { return gd.n[0] > 1; }

// exclusive scan of the histogram in c->cursor -> out (and cursor := out)
int run_scan(psc_ctx *c, int32_t *out, cudaStream_t s) {
  const int nk = c->gd.nkeys;
  ProfScope ps(c, PSC_PH_SORT_SCAN, s);
  const int sblocks = (int)cdiv64(nk, SCAN_TILE);
  int *tmp = (int *)c->scan_tmp;
  k_scan_local<int><<<sblocks, SORT_THREADS, 0, s>>>(nk, c->cursor, out, tmp);
  PSC_LAUNCH_CHECK(c);
  k_scan_tmp<int><<<1, 1024, 0, s>>>(sblocks, tmp);
  PSC_LAUNCH_CHECK(c);
  k_scan_add<<<sblocks, SORT_THREADS, 0, s>>>(nk, out, c->cursor, tmp, sblocks);
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}

// packed scan of c->pack -> out_hi (cell offsets), out_lo (arrival-list offsets)
int run_scan2(psc_ctx *c, int32_t *out_hi, int32_t *out_lo, cudaStream_t s) {
  const int nk = c->gd.nkeys;
  ProfScope ps(c, PSC_PH_SORT_SCAN, s);
  const int sblocks = (int)cdiv64(nk, SCAN_TILE);
  k_scan_local<long long><<<sblocks, SORT_THREADS, 0, s>>>(nk, c->pack, c->packloc, c->scan_tmp);
  PSC_LAUNCH_CHECK(c);
  k_scan_tmp<long long><<<1, 1024, 0, s>>>(sblocks, c->scan_tmp);
  PSC_LAUNCH_CHECK(c);
  k_scan_add2<<<sblocks, SORT_THREADS, 0, s>>>(nk, c->packloc, out_hi, out_lo, c->scan_tmp, sblocks);
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}

// key[s] of the particles of the current column set, in their current order
int slot_keys(psc_ctx *c, int32_t *key, cudaStream_t s) {
  const int n = (int)c->np;
  if (n == 0) return PSC_OK;
  const int32_t *offs, *dirtab = nullptr;
  switch (c->state) {
    case PSC_STATE_SORTED: offs = c->offs[c->ocur]; break;
    case PSC_STATE_PUSHED: offs = c->offs[c->ocur]; dirtab = c->dircnt; break;
    case PSC_STATE_INDEXED: offs = c->offs[c->ocur ^ 1]; dirtab = c->dircnt; break;
    default: return PSC_ERR_NOT_SORTED;
  }
  const int blocks = (int)cdiv64(n, SORT_THREADS);
  if (is3d(c->gd)) k_slot_keys<true><<<blocks, SORT_THREADS, 0, s>>>(c->gd, n, offs, dirtab, c->dcode, key);
  else k_slot_keys<false><<<blocks, SORT_THREADS, 0, s>>>(c->gd, n, offs, dirtab, c->dcode, key);
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}

}  // namespace

// key[] (c->curkey) := keys of the current particles, in their current order
int psc_sort_current_keys(psc_ctx *c, cudaStream_t s) { return slot_keys(c, c->curkey, s); }

// general counting sort: arbitrary order in, physically sorted (stable) list out
int psc_sort_general(psc_ctx *c, cudaStream_t s) {
  const GridDesc &gd = c->gd;
  const int n = (int)c->np;
  const int nk = gd.nkeys;
  const Cols &in = c->cols[c->cur];
  const Cols &out = c->cols[c->cur ^ 1];
  const int pblocks = (int)min((int64_t)c->sm_count * 16, max((int64_t)1, cdiv64(n, SORT_THREADS)));

  if (c->form == PSC_FORM_REL) {  // a sorted or pushed list sorted again: keys from the slots
    const int rc = slot_keys(c, c->key, s);
    if (rc) return rc;
    if (c->state == PSC_STATE_INDEXED) c->ocur ^= 1;  // back to the layout of the written list
  }
  int32_t *offs_new = c->offs[c->ocur ^ 1];
  PSC_CUDA_TRY(c, cudaMemsetAsync(c->cursor, 0, (size_t)(nk + 1) * 4, s));
  PSC_CUDA_TRY(c, cudaMemsetAsync(c->d_flags + 1, 0, 4, s));
  c->launches += 2;
  psc_prof_begin(c, PSC_PH_SORT_COUNT, s);
  if (c->form == PSC_FORM_ABS)
    k_keys<<<pblocks, SORT_THREADS, 0, s>>>(gd, n, in.x, in.y, in.z, c->key, c->cursor, c->d_flags);
  else
    k_hist<<<pblocks, SORT_THREADS, 0, s>>>(n, nk, c->key, c->cursor, c->d_flags);
  PSC_LAUNCH_CHECK(c);
  psc_prof_end(c, PSC_PH_SORT_COUNT, s);
  {
    const int rc = run_scan(c, offs_new, s);
    if (rc) return rc;
  }
  psc_prof_begin(c, PSC_PH_SORT_RANK, s);
  k_scatter<<<pblocks, SORT_THREADS, 0, s>>>(n, c->key, c->cursor, c->perm);
  PSC_LAUNCH_CHECK(c);
  const int kblocks = (int)min((int64_t)c->sm_count * 8, max((int64_t)1, cdiv64(nk, SORT_THREADS / 32)));
  k_segsort<<<kblocks, SORT_THREADS, 0, s>>>(nk, offs_new, c->perm, c->big_list, c->d_flags + 1);
  PSC_LAUNCH_CHECK(c);
  if (n > WARP_SEG_CAP) {
    static bool attr_set = false;
    if (!attr_set) {
      PSC_CUDA_TRY(c, cudaFuncSetAttribute(k_segsort_big, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           BIG_SMEM_CAP * 4));
      attr_set = true;
    }
    k_segsort_big<<<c->sm_count, 1024, BIG_SMEM_CAP * 4, s>>>(offs_new, c->perm, c->big_list,
                                                              c->d_flags + 1);
    PSC_LAUNCH_CHECK(c);
  }
  psc_prof_end(c, PSC_PH_SORT_RANK, s);
  psc_prof_begin(c, PSC_PH_SORT_REORDER, s);
  if (c->form == PSC_FORM_ABS) k_reorder<true><<<pblocks, SORT_THREADS, 0, s>>>(gd, n, c->perm, in, out);
  else k_reorder<false><<<pblocks, SORT_THREADS, 0, s>>>(gd, n, c->perm, in, out);
  PSC_LAUNCH_CHECK(c);
  psc_prof_end(c, PSC_PH_SORT_REORDER, s);
  c->cur ^= 1;
  c->ocur ^= 1;
  c->form = PSC_FORM_REL;
  c->state = PSC_STATE_SORTED;
  c->have_sort_result = 1;
  return PSC_OK;
}

// index sort of a pushed list: new cell offsets + the arrival list from the per-cell direction
// counts and the leavers' direction codes; no column moves
int psc_sort_index(psc_ctx *c, cudaStream_t s) {
  const GridDesc &gd = c->gd;
  const int nk = gd.nkeys;
  const int32_t *offs_w = c->offs[c->ocur];  // layout of the written list
  int32_t *offs_new = c->offs[c->ocur ^ 1];
  const int cblocks = (int)cdiv64(nk, SORT_THREADS);
  const bool d3 = is3d(gd);
  psc_prof_begin(c, PSC_PH_SORT_COUNT, s);
  if (d3) k_dest_hist<true><<<cblocks, SORT_THREADS, 0, s>>>(gd, c->dircnt, c->nstay, c->pack);
  else k_dest_hist<false><<<cblocks, SORT_THREADS, 0, s>>>(gd, c->dircnt, c->nstay, c->pack);
  PSC_LAUNCH_CHECK(c);
  psc_prof_end(c, PSC_PH_SORT_COUNT, s);
  {
    const int rc = run_scan2(c, offs_new, c->aoffs, s);
    if (rc) return rc;
  }
  psc_prof_begin(c, PSC_PH_SORT_RANK, s);
  if (d3) k_dir_base<true><<<cblocks, SORT_THREADS, 0, s>>>(gd, c->dircnt, c->aoffs);
  else k_dir_base<false><<<cblocks, SORT_THREADS, 0, s>>>(gd, c->dircnt, c->aoffs);
  PSC_LAUNCH_CHECK(c);
  const int rblocks = (int)min((int64_t)c->sm_count * 32, max((int64_t)1, cdiv64(nk, (SORT_THREADS / 32) * 4)));
  if (d3) k_rank<true><<<rblocks, SORT_THREADS, 0, s>>>(nk, offs_w, c->dcode, c->dircnt, c->alist, c->d_flags);
  else k_rank<false><<<rblocks, SORT_THREADS, 0, s>>>(nk, offs_w, c->dcode, c->dircnt, c->alist, c->d_flags);
  PSC_LAUNCH_CHECK(c);
  psc_prof_end(c, PSC_PH_SORT_RANK, s);
  c->ocur ^= 1;
  c->state = PSC_STATE_INDEXED;
  c->have_sort_result = 0;
  return PSC_OK;
}

// cell_idx[a] of the last (general) sort's INPUT particles
int psc_sort_cell_idx(psc_ctx *c, cudaStream_t s) {
  const int n = (int)c->np;
  if (n == 0) return PSC_OK;
  k_cell_idx<<<(int)cdiv64(n, SORT_THREADS), SORT_THREADS, 0, s>>>(c->gd, n, c->key, c->cell_idx);
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}

int psc_particles_to_abs(psc_ctx *c, cudaStream_t s) {
  const int n = (int)c->np;
  if (n) {
    const int rc = psc_sort_current_keys(c, s);
    if (rc) return rc;
    const Cols &p = c->cols[c->cur];
    k_to_abs<<<(int)cdiv64(n, SORT_THREADS), SORT_THREADS, 0, s>>>(c->gd, n, c->curkey, p.x, p.y, p.z);
    PSC_LAUNCH_CHECK(c);
  }
  c->form = PSC_FORM_ABS;
  c->state = PSC_STATE_UNSORTED;
  c->have_sort_result = 0;
  return PSC_OK;
}
