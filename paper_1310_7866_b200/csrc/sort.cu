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
// advanced by one push, which left per particle a one-byte direction code (one of 9 / 27
// destination classes) and per cell the count of each code.  Then
//   1. k_dest_hist  new count of cell k = sum over its 9 / 27 neighbour source cells of the
//                   count of the code that points at k;
//   2. scan         -> new cell offsets;
//   3. k_dir_base   stable order inside a destination cell = ascending old slot = ascending
//                   source-cell key, then slot order inside the source cell: first slot of every
//                   (source cell, code) group by a running sum over the sources in key order;
//   4. k_rank       one warp per source cell walks its slots in order and hands out
//                   consecutive slots per code (ballot + popc for the stayers, lane order for the
//                   few leavers) -> perm.  Reads 1 byte, writes 4 bytes per particle.
// No particle column is touched: the next push loads particle perm[s] for slot s (reorder on
// load).  psc_particles_sort, whose contract is a physically sorted list, adds k_reorder.
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
    float v = ((float)c[d] + pos[d][a]) * gd.dx[d];
    if (v >= gd.L[d]) v = nextafterf(gd.L[d], 0.f);  // rounding must not leave [0, L)
    pos[d][a] = v;
  }
}

// ---- exclusive scan of hist[0..m) -> out[0..m], out[m] = total; also cursor := out -----------

__global__ void __launch_bounds__(SORT_THREADS)
k_scan_local(int m, const int *__restrict__ in, int *__restrict__ out, int *__restrict__ tmp) {
  __shared__ int wsum[SORT_THREADS / 32];
  const int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  int v[SCAN_ITEMS];
  int s = 0;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++) {
    v[i] = (base + i < m) ? in[base + i] : 0;
    s += v[i];
  }
  // inclusive scan of s across the block
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int inc = s;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) wsum[w] = inc;
  __syncthreads();
  if (w == 0) {
    int t = lane < SORT_THREADS / 32 ? wsum[lane] : 0;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, t, o);
      if (lane >= o) t += u;
    }
    if (lane < SORT_THREADS / 32) wsum[lane] = t;
  }
  __syncthreads();
  int run = inc - s + (w ? wsum[w - 1] : 0);
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++) {
    if (base + i < m) out[base + i] = run;
    run += v[i];
  }
  if (threadIdx.x == SORT_THREADS - 1) tmp[blockIdx.x] = run;
}

// single block: exclusive scan of tmp[0..nb) in place, tmp[nb] = total
__global__ void __launch_bounds__(1024) k_scan_tmp(int nb, int *__restrict__ tmp) {
  __shared__ int wsum[32];
  __shared__ int carry_s;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int base = 0; base < nb; base += 1024) {
    const int i = base + threadIdx.x;
    const int v = i < nb ? tmp[i] : 0;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    if (w == 0) {
      int t = wsum[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int u = __shfl_up_sync(0xffffffffu, t, o);
        if (lane >= o) t += u;
      }
      wsum[lane] = t;
    }
    __syncthreads();
    const int carry = carry_s;
    const int exc = carry + inc - v + (w ? wsum[w - 1] : 0);
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
    if (FROM_ABS) {  // same fp32 product + floor as k_keys; clamped like there
      if (gd.n[0] > 1) { const float xi = __fmul_rn(x, gd.inv_dx[0]); x = fminf(fmaxf(xi - floorf(xi), 0.f), 0.99999994f); }
      if (gd.n[1] > 1) { const float xi = __fmul_rn(y, gd.inv_dx[1]); y = fminf(fmaxf(xi - floorf(xi), 0.f), 0.99999994f); }
      if (gd.n[2] > 1) { const float xi = __fmul_rn(z, gd.inv_dx[2]); z = fminf(fmaxf(xi - floorf(xi), 0.f), 0.99999994f); }
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

// key of the neighbour of cell c[] in direction code dc (periodic)
template <bool D3>
__device__ __forceinline__ int neighbour_key(const GridDesc &gd, const int c[3], int dc, int sign) {
  int s[3];
  if (D3) {
    s[0] = dc % 3 - 1;
    s[1] = (dc / 3) % 3 - 1;
    s[2] = dc / 9 - 1;
  } else {
    s[0] = 0;
    s[1] = dc % 3 - 1;
    s[2] = dc / 3 - 1;
  }
  int q[3];
#pragma unroll
  for (int d = 0; d < 3; d++) q[d] = wrap(c[d] + sign * s[d], gd.n[d]);
  return cell_to_key(gd, q);
}

// hist[k] = particles that will be in cell k: source cell (k - dir) sends count[dir]
template <bool D3>
__global__ void __launch_bounds__(SORT_THREADS)
k_dest_hist(GridDesc gd, const int *__restrict__ dircnt, int *__restrict__ hist) {
  constexpr int ND = D3 ? 27 : 9;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= gd.nkeys) return;
  int c[3];
  key_to_cell(gd, k, c);
  int tot = 0;
#pragma unroll
  for (int dc = 0; dc < ND; dc++) tot += dircnt[neighbour_key<D3>(gd, c, dc, -1) * ND + dc];
  hist[k] = tot;
}

// dircnt[src][dc] (count) -> first new slot of the (src, dc) group, in place
template <bool D3>
__global__ void __launch_bounds__(SORT_THREADS)
k_dir_base(GridDesc gd, int *__restrict__ dircnt, const int *__restrict__ offs_new) {
  constexpr int ND = D3 ? 27 : 9;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= gd.nkeys) return;
  int c[3];
  key_to_cell(gd, k, c);
  int sk[ND], cnt[ND];
#pragma unroll
  for (int dc = 0; dc < ND; dc++) {
    sk[dc] = neighbour_key<D3>(gd, c, dc, -1);
    cnt[dc] = dircnt[sk[dc] * ND + dc];
  }
  const int o = offs_new[k];
#pragma unroll
  for (int i = 0; i < ND; i++) {
    int b = o;
#pragma unroll
    for (int j = 0; j < ND; j++) b += (sk[j] < sk[i]) ? cnt[j] : 0;
    dircnt[sk[i] * ND + i] = b;
  }
}

// one warp per source cell: perm[new slot] = old slot
template <bool D3>
__global__ void __launch_bounds__(SORT_THREADS)
k_rank(int nkeys, const int *__restrict__ offs_old, const uint8_t *__restrict__ dcode,
       const int *__restrict__ dirbase, int *__restrict__ perm, uint32_t *__restrict__ flags) {
  constexpr int ND = D3 ? 27 : 9, STAY = D3 ? 13 : 4;
  __shared__ int sb[SORT_THREADS / 32][32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int warps = gridDim.x * (SORT_THREADS / 32);
  const unsigned lt = lanemask_lt();
  for (int k = blockIdx.x * (SORT_THREADS / 32) + w; k < nkeys; k += warps) {
    const int p0 = offs_old[k], p1 = offs_old[k + 1];
    if (p0 >= p1) continue;
    const int b = lane < ND ? dirbase[k * ND + lane] : 0;
    sb[w][lane] = b;
    int bstay = __shfl_sync(0xffffffffu, b, STAY);
    __syncwarp();
    for (int base = p0; base < p1; base += 32) {
      const int s = base + lane;
      const bool act = s < p1;
      int dc = act ? (int)dcode[s] : STAY;
      if (dc >= ND) {  // cannot happen unless the caller scribbled over the workspace
        atomicOr(flags, PSC_F_OOB);
        dc = STAY;
      }
      const bool stay = act && dc == STAY;
      const unsigned m = __ballot_sync(0xffffffffu, stay);
      int slot = bstay + __popc(m & lt);
      bstay += __popc(m);
      unsigned lv = __ballot_sync(0xffffffffu, act && !stay);
      while (lv) {  // the few leavers, in lane order (= slot order: stable)
        const int l = __ffs(lv) - 1;
        lv &= lv - 1;
        if (lane == l) {
          slot = sb[w][dc];
          sb[w][dc] = slot + 1;
        }
        __syncwarp();
      }
      if (act) perm[slot] = s;
    }
    __syncwarp();
  }
}

// key of the particle in slot s of a list laid out by `offs`: the slot's cell, moved by the
// particle's direction code if there is one
template <bool D3>
__global__ void __launch_bounds__(SORT_THREADS)
k_slot_keys(GridDesc gd, int n, const int *__restrict__ offs, const uint8_t *__restrict__ dcode,
            int *__restrict__ key) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  int lo = 0, hi = gd.nkeys;  // largest k with offs[k] <= s (and offs[k+1] > s)
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (offs[mid] <= s) lo = mid; else hi = mid;
  }
  int k = lo;
  if (dcode) {
    int c[3];
    key_to_cell(gd, k, c);
    k = neighbour_key<D3>(gd, c, (int)dcode[s], +1);
  }
  key[s] = k;
}

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace

size_t psc_sort_workspace_bytes(const psc_ctx *c, int64_t n) {
  const size_t nk = (size_t)c->gd.nkeys;
  size_t b = 0;
  b += 4 * align_up((size_t)n * 4, 256);                      // key, perm, cell_idx, curkey
  b += align_up((size_t)n, 256);                              // dcode
  b += 3 * align_up((nk + 1) * 4, 256);                       // offs[2], cursor
  b += align_up(nk * 27 * 4, 256);                            // dircnt
  b += align_up((nk / SCAN_TILE + 3) * 4, 256);               // scan_tmp
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
  c->dcode = (uint8_t *)take((size_t)n);
  c->offs[0] = (int32_t *)take((nk + 1) * 4);
  c->offs[1] = (int32_t *)take((nk + 1) * 4);
  c->cursor = (int32_t *)take((nk + 1) * 4);
  c->dircnt = (int32_t *)take(nk * 27 * 4);
  c->scan_tmp = (int32_t *)take((nk / SCAN_TILE + 3) * 4);
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
  k_scan_local<<<sblocks, SORT_THREADS, 0, s>>>(nk, c->cursor, out, c->scan_tmp);
  PSC_LAUNCH_CHECK(c);
  k_scan_tmp<<<1, 1024, 0, s>>>(sblocks, c->scan_tmp);
  PSC_LAUNCH_CHECK(c);
  k_scan_add<<<sblocks, SORT_THREADS, 0, s>>>(nk, out, c->cursor, c->scan_tmp, sblocks);
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}

int slot_keys(psc_ctx *c, const int32_t *offs, const uint8_t *dcode, int32_t *key, cudaStream_t s) {
  const int n = (int)c->np;
  if (n == 0) return PSC_OK;
  const int blocks = (int)cdiv64(n, SORT_THREADS);
  if (is3d(c->gd)) k_slot_keys<true><<<blocks, SORT_THREADS, 0, s>>>(c->gd, n, offs, dcode, key);
  else k_slot_keys<false><<<blocks, SORT_THREADS, 0, s>>>(c->gd, n, offs, dcode, key);
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}

}  // namespace

// key[] (c->curkey) := keys of the current particles, in their current order
int psc_sort_current_keys(psc_ctx *c, cudaStream_t s) {
  switch (c->state) {
    case PSC_STATE_SORTED: return slot_keys(c, c->offs[c->ocur], nullptr, c->curkey, s);
    case PSC_STATE_PUSHED: return slot_keys(c, c->offs[c->ocur], c->dcode, c->curkey, s);
    case PSC_STATE_INDEXED: return slot_keys(c, c->offs[c->ocur ^ 1], c->dcode, c->curkey, s);
    default: return PSC_ERR_NOT_SORTED;
  }
}

// general counting sort: arbitrary order in, physically sorted list out
int psc_sort_general(psc_ctx *c, cudaStream_t s) {
  const GridDesc &gd = c->gd;
  const int n = (int)c->np;
  const int nk = gd.nkeys;
  const Cols &in = c->cols[c->cur];
  const Cols &out = c->cols[c->cur ^ 1];
  const int pblocks = (int)min((int64_t)c->sm_count * 16, max((int64_t)1, cdiv64(n, SORT_THREADS)));
  int32_t *offs_new = c->offs[c->ocur ^ 1];

  if (c->form == PSC_FORM_REL) {  // a sorted list sorted again: keys from the slots
    const int rc = slot_keys(c, c->offs[c->ocur], nullptr, c->key, s);
    if (rc) return rc;
  }
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

// index sort of a pushed list: new offsets + perm from the direction codes; no column moves
int psc_sort_index(psc_ctx *c, cudaStream_t s) {
  const GridDesc &gd = c->gd;
  const int nk = gd.nkeys;
  const int32_t *offs_old = c->offs[c->ocur];
  int32_t *offs_new = c->offs[c->ocur ^ 1];
  const int cblocks = (int)cdiv64(nk, SORT_THREADS);
  const bool d3 = is3d(gd);
  psc_prof_begin(c, PSC_PH_SORT_COUNT, s);
  if (d3) k_dest_hist<true><<<cblocks, SORT_THREADS, 0, s>>>(gd, c->dircnt, c->cursor);
  else k_dest_hist<false><<<cblocks, SORT_THREADS, 0, s>>>(gd, c->dircnt, c->cursor);
  PSC_LAUNCH_CHECK(c);
  psc_prof_end(c, PSC_PH_SORT_COUNT, s);
  {
    const int rc = run_scan(c, offs_new, s);
    if (rc) return rc;
  }
  psc_prof_begin(c, PSC_PH_SORT_RANK, s);
  if (d3) k_dir_base<true><<<cblocks, SORT_THREADS, 0, s>>>(gd, c->dircnt, offs_new);
  else k_dir_base<false><<<cblocks, SORT_THREADS, 0, s>>>(gd, c->dircnt, offs_new);
  PSC_LAUNCH_CHECK(c);
  const int rblocks = (int)min((int64_t)c->sm_count * 32, max((int64_t)1, cdiv64(nk, SORT_THREADS / 32)));
  if (d3) k_rank<true><<<rblocks, SORT_THREADS, 0, s>>>(nk, offs_old, c->dcode, c->dircnt, c->perm, c->d_flags);
  else k_rank<false><<<rblocks, SORT_THREADS, 0, s>>>(nk, offs_old, c->dcode, c->dircnt, c->perm, c->d_flags);
  PSC_LAUNCH_CHECK(c);
  psc_prof_end(c, PSC_PH_SORT_RANK, s);
  c->ocur ^= 1;
  c->state = PSC_STATE_INDEXED;
  c->have_sort_result = 2;
  return PSC_OK;
}

// INDEXED -> SORTED: the physical reorder the next push would otherwise do on load
int psc_sort_materialize(psc_ctx *c, cudaStream_t s) {
  const int n = (int)c->np;
  const int pblocks = (int)min((int64_t)c->sm_count * 16, max((int64_t)1, cdiv64(n, SORT_THREADS)));
  ProfScope ps(c, PSC_PH_SORT_REORDER, s);
  k_reorder<false><<<pblocks, SORT_THREADS, 0, s>>>(c->gd, n, c->perm, c->cols[c->cur], c->cols[c->cur ^ 1]);
  PSC_LAUNCH_CHECK(c);
  c->cur ^= 1;
  c->state = PSC_STATE_SORTED;
  return PSC_OK;
}

// cell_idx[a] of the last sort's INPUT particles
int psc_sort_cell_idx(psc_ctx *c, cudaStream_t s) {
  const int n = (int)c->np;
  if (n == 0) return PSC_OK;
  if (c->have_sort_result == 2) {  // index sort: input key = old slot's cell moved by the code
    const int rc = slot_keys(c, c->offs[c->ocur ^ 1], c->dcode, c->key, s);
    if (rc) return rc;
  }
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
