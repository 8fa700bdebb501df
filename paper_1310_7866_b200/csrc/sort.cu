// sort.cu -- cell-key counting sort of the particle list and the layout of
// the cell store it produces.
//
// One key orders by block ("supercell") and by cell inside the block at once:
//   key = block_index * cells_per_block + cell_in_block.
// A counting sort is O(N + M):
//   1. k_keys     key per particle from floor(fl32(x * 1/dx)) (k_hist: keys already known), and a
//                 histogram over keys with warp-aggregated atomics;
//   2. k_layout   capacity of every cell = its count plus spare room, rounded up to 32 slots;
//      scan       one exclusive prefix sum over (capacity, count) packed in 64 bits -> the first
//                 slot base[k] of every cell in the store and the dense offsets of the sorted list;
//   3. k_scatter  dense position = cursor[key] + rank, again warp-aggregated; writes the permutation;
//   4. k_segsort  the atomics hand out positions in arbitrary order ACROSS warps, so every key's
//                 segment of `perm` is sorted ascending: a set of distinct input indices in
//                 ascending order IS the stable order, hence the result is the unique stable
//                 counting sort, bit-exact against any stable reference;
//   5. k_reorder  out[base[k] + rank] = in[perm[s]] for every column; positions leave in the
//                 internal form (in-cell offsets).
//
// PAPER.md:597-603 ("a particle moves at most one cell per step", "reorder on load"): between
// pushes NO sort runs.  The push kernels keep every cell's particles dense in the cell's own
// slots and hand the few cell-changers over through the exchange rows (store.cuh).  Only when a
// push had to spill (an exchange row or a cell ran out of room) something happens between two
// pushes: k_spill_insert files the spilled particles straight into their destination cells where
// these have a free slot; if some are left (cells that are really full) the store is re-laid out:
// k_tot / scan / k_gather flatten residents + exchange records + spill list into the other
// column set, and steps 1-5 (without 4: the order inside a cell is immaterial, A17)
// bring them back.  Whether any of that is needed is known on the device only: one gate kernel
// looks at the spill counter and launches the rest from the device.
#include <limits.h>
#include <math.h>

#include "store.cuh"

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

#define PSC_COND_RETURN(cond) \
  if ((cond) && !*(cond)) return

__global__ void __launch_bounds__(SORT_THREADS)
k_keys(GridDesc gd, int n, const float *__restrict__ x, const float *__restrict__ y,
       const float *__restrict__ z, const int *__restrict__ sp, int *__restrict__ key,
       int *__restrict__ hist, uint32_t *__restrict__ flags) {
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
        // a product that rounds up to n although x < L belongs to the last cell (its offset is
        // then clamped just below 1 by k_reorder): not a fault
        if (ci == gd.n[d] && pos[d][a] < gd.L[d]) ci = gd.n[d] - 1;
        if (!(ci >= 0 && ci < gd.n[d])) {  // also catches NaN
          oob = true;
          ci = ci < 0 ? 0 : gd.n[d] - 1;
          if (xi != xi) ci = 0;
        }
        c[d] = ci;
      }
      if (oob) atomicOr(flags, PSC_F_OOB);
      const int s = sp[a];
      if (s < 0 || s >= gd.nsp) atomicOr(flags, PSC_F_SPECIES);
      k = cell_key(gd, c[0], c[1], c[2]);
      key[a] = k;
    }
    const unsigned grp = __match_any_sync(0xffffffffu, k);
    if (valid && (grp & lanemask_lt()) == 0) atomicAdd(&hist[k], __popc(grp));
  }
}

// histogram of keys that already exist (a flattened store)
__global__ void __launch_bounds__(SORT_THREADS)
k_hist(const int *__restrict__ np, int nkeys, const int *__restrict__ key, int *__restrict__ hist,
       uint32_t *__restrict__ flags, const uint32_t *__restrict__ cond) {
  PSC_COND_RETURN(cond);
  const int n = *np;
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

__global__ void __launch_bounds__(SORT_THREADS)
k_zero(int m, int *__restrict__ a, const uint32_t *__restrict__ cond) {
  PSC_COND_RETURN(cond);
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < m; i += gridDim.x * blockDim.x) a[i] = 0;
}

__global__ void __launch_bounds__(SORT_THREADS)
k_cell_idx(GridDesc gd, int n, const int *__restrict__ key, int *__restrict__ cell_idx) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n) return;
  int c[3];
  key_to_cell(gd, key[a], c);
  cell_idx[a] = (c[2] * gd.n[1] + c[1]) * gd.n[0] + c[0];
}

// Capacity of a cell holding cnt particles: room for an eighth more, and at least for six
// standard deviations of a Poisson count (the population of a cell of a uniform plasma fluctuates
// by sqrt(cnt); with millions of cells some reach +5 sigma within a few steps), rounded up to a
// multiple of 32 slots so that every column of every cell starts on a 128-byte line.
// Sum over cells <= n + n/8 + 6 sqrt(nkeys n) + 56 nkeys (psc_store_capacity; Cauchy-Schwarz).
__host__ __device__ __forceinline__ int cell_capacity(int cnt) {
  const int sig = (int)(6.0f * sqrtf((float)cnt)) + 8;
  const int spare = max(max(cnt >> 3, 16), sig);
  return (cnt + spare + PSC_SLOT_ALIGN - 1) & ~(PSC_SLOT_ALIGN - 1);
}

// per cell: pack = capacity << 32 | count for the packed scan; cnt := count; stats: largest count
__global__ void __launch_bounds__(SORT_THREADS)
k_layout(int nk, const int *__restrict__ hist, long long *__restrict__ pack, int *__restrict__ cnt,
         uint32_t *__restrict__ dw, const uint32_t *__restrict__ cond) {
  PSC_COND_RETURN(cond);
  int mx = 0;
  for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < nk; k += gridDim.x * blockDim.x) {
    const int c = hist[k];
    cnt[k] = c;
    pack[k] = ((long long)cell_capacity(c) << 32) | (long long)c;
    mx = max(mx, c);
  }
#pragma unroll
  for (int o = 16; o; o >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if ((threadIdx.x & 31) == 0 && mx) atomicMax(&dw[PSC_DW_MAXCNT], (uint32_t)mx);
}

// ---- exclusive scan of in[0..m) -> out[0..m], out[m] = total -----------------------------------
// T = int: one histogram (cursor := out as well if given).  T = long long: two histograms packed
// as (hi << 32) | lo and scanned in one pass (the layout: hi = capacity of a cell, lo = particles
// in it; both totals are < 2^31, so the low half never carries into the high half); the last
// kernel unpacks them into out (hi) and out_lo.
// cond != nullptr: the launch does nothing unless *cond != 0 (a re-layout only runs when the
// previous push spilled; the host cannot know without synchronising, so the device decides).

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
k_scan_local(int m, const T *__restrict__ in, T *__restrict__ out, T *__restrict__ tmp,
             const uint32_t *__restrict__ cond) {
  if (cond && !*cond) return;
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
__global__ void __launch_bounds__(1024) k_scan_tmp(int nb, T *__restrict__ tmp, const uint32_t *__restrict__ cond) {
  if (cond && !*cond) return;
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
           int nb, const uint32_t *__restrict__ cond) {
  if (cond && !*cond) return;
  const int add = tmp[blockIdx.x];
  const int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++)
    if (base + i < m) {
      const int v = out[base + i] + add;
      out[base + i] = v;
      if (cursor) cursor[base + i] = v;
    }
  if (blockIdx.x == 0 && threadIdx.x == 0) out[m] = tmp[nb];
}

// packed form: loc[] holds the block-local packed scan; out := high halves, out_lo := low halves
__global__ void __launch_bounds__(SORT_THREADS)
k_scan_add2(int m, const long long *__restrict__ loc, int *__restrict__ out,
            int *__restrict__ out_lo, int *__restrict__ cursor, const long long *__restrict__ tmp, int nb,
            const uint32_t *__restrict__ cond) {
  if (cond && !*cond) return;
  const long long add = tmp[blockIdx.x];
  const int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++)
    if (base + i < m) {
      const long long v = loc[base + i] + add;
      out[base + i] = (int)(v >> 32);
      out_lo[base + i] = (int)(v & 0xffffffffLL);
      cursor[base + i] = (int)(v & 0xffffffffLL);
    }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    out[m] = (int)(tmp[nb] >> 32);
    out_lo[m] = (int)(tmp[nb] & 0xffffffffLL);
  }
}

__global__ void __launch_bounds__(SORT_THREADS)
k_scatter(const int *__restrict__ np, const int *__restrict__ key, int *__restrict__ cursor,
          int *__restrict__ perm, const uint32_t *__restrict__ cond) {
  PSC_COND_RETURN(cond);
  const int n = *np;
  const int lane = threadIdx.x & 31;
  // Every warp walks ONE contiguous span of the input, 32 particles at a time: a key whose
  // particles all lie inside one span (a list that is already ordered by cell, e.g. as generated
  // or after a few pushes) gets its positions in ascending input order, and k_segsort finds its
  // segment already sorted.  (Spans are multiples of 32, so every load is a full 128-byte line.)
  const long long nwarps = (long long)gridDim.x * (blockDim.x >> 5);
  const long long wid = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const long long span = ((n + nwarps - 1) / nwarps + 31) / 32 * 32;
  const long long lo = wid * span, hi = lo + span < n ? lo + span : n;
  for (long long a = lo + lane; a - lane < hi; a += 32) {
    const bool valid = a < hi;
    const int k = valid ? key[a] : -1 - lane;
    const unsigned grp = __match_any_sync(0xffffffffu, k);
    const int leader = __ffs(grp) - 1;
    int base = 0;
    if (valid && lane == leader) base = atomicAdd(&cursor[k], __popc(grp));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (valid) perm[base + __popc(grp & lanemask_lt())] = (int)a;
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

// Sorted position s holds input particle perm[s]; its cell k = key[perm[s]] starts at dense
// offset offs[k] and at slot base[k] of the store.  FROM_ABS: the input columns hold absolute
// positions -> write in-cell offsets.
template <bool FROM_ABS>
__global__ void __launch_bounds__(SORT_THREADS)
k_reorder(GridDesc gd, const int *__restrict__ np, const int *__restrict__ perm,
          const int *__restrict__ key, const int *__restrict__ offs, const int *__restrict__ base,
          Cols in, Cols out, const uint32_t *__restrict__ cond) {
  PSC_COND_RETURN(cond);
  const int n = *np;
  const int s0 = blockIdx.x * blockDim.x + threadIdx.x;
  const int stride = gridDim.x * blockDim.x;
  for (int s = s0; s < n; s += stride) {
    const int p = perm[s];
    const int k = key[p];
    const size_t o = (size_t)base[k] + (s - offs[k]);
    float x = in.x ? in.x[p] : 0.f, y = in.y[p], z = in.z[p];
    const float ux = in.ux[p], uy = in.uy[p], uz = in.uz[p];
    const float qw = in.qw[p];
    int sp = in.sp[p];
    int id = 0;
    if (in.id) id = in.id[p];
    if (FROM_ABS) {
      // the cell is the one k_keys decided (key[p]); the offset is (x - cell dx) / dx with the
      // difference formed by one FMA, i.e. accurate to fp32 RELATIVE precision of the offset also
      // when dx is not a power of two (x * (1/dx) - cell would carry the absolute rounding error
      // of x / dx, ~1e-6 cells at x / dx ~ 20)
      int c[3];
      key_to_cell(gd, k, c);
      auto rel = [&](float v, int d) {
        return fminf(fmaxf(fmaf(-(float)c[d], gd.dx[d], v) * gd.inv_dx[d], 0.f), 0.99999994f);
      };
      if (gd.n[0] > 1) x = rel(x, 0);
      if (gd.n[1] > 1) y = rel(y, 1);
      if (gd.n[2] > 1) z = rel(z, 2);
      if (sp < 0 || sp >= gd.nsp) sp = 0;  // flagged by k_keys (PSC_F_SPECIES)
    }
    if (in.x) out.x[o] = x;
    out.y[o] = y;
    out.z[o] = z;
    out.ux[o] = ux;
    out.uy[o] = uy;
    out.uz[o] = uz;
    out.qw[o] = qw;
    out.sp[o] = sp;
    if (in.id) out.id[o] = id;
  }
}

// ---- flattening the store -----------------------------------------------------------------------

// records waiting in the exchange row of cell k: the union of its per-direction masks
__device__ __forceinline__ unsigned row_union(const uint32_t *__restrict__ mask, int k, int xw, int nd) {
  unsigned u = 0;
  for (int d = 0; d < nd; d++) u |= mask[(size_t)k * xw + d];
  return u;
}

// tot[k] = residents of cell k + records waiting in its exchange row
__global__ void __launch_bounds__(SORT_THREADS)
k_tot(int nk, int xw, int nd, const int *__restrict__ cnt, const uint32_t *__restrict__ mask,
      int *__restrict__ tot, const uint32_t *__restrict__ cond) {
  PSC_COND_RETURN(cond);
  for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < nk; k += gridDim.x * blockDim.x)
    tot[k] = cnt[k] + __popc(row_union(mask, k, xw, nd));
}

// A warp per cell copies the cell's residents, then the records of its exchange row, to the dense
// positions doffs[k] ...; key = the cell the offsets refer to (for a record: the destination of
// its move).  ABS: positions become x = (cell + offset) * dx, formed in fp64 and rounded once.
template <bool D3, bool ABS>
__global__ void __launch_bounds__(SORT_THREADS)
k_gather(GridDesc gd, Cols in, const int *__restrict__ base, const int *__restrict__ cnt,
         Exchange xin, const int *__restrict__ doffs, Cols out, int *__restrict__ keyout,
         const uint32_t *__restrict__ cond) {
  PSC_COND_RETURN(cond);
  const int lane = threadIdx.x & 31;
  const int warps = gridDim.x * (SORT_THREADS / 32);
  for (int k = blockIdx.x * (SORT_THREADS / 32) + (threadIdx.x >> 5); k < gd.nkeys; k += warps) {
    const int n = cnt[k], d0 = doffs[k], nt = doffs[k + 1] - d0;
    if (nt == 0) continue;
    int c[3];
    key_to_cell(gd, k, c);
    auto absf = [&](float off, int cell, int d) {
      float v = __double2float_rn(((double)cell + (double)off) * (double)gd.dx[d]);
      if (v >= gd.L[d]) v = nextafterf(gd.L[d], 0.f);  // rounding must not leave [0, L)
      return v;
    };
    const size_t b = (size_t)base[k];
    for (int i = lane; i < n; i += 32) {
      const size_t s = b + i, o = (size_t)d0 + i;
      float x = in.x ? in.x[s] : 0.f, y = in.y[s], z = in.z[s];
      if (ABS) {
        if (D3) x = absf(x, c[0], 0);
        y = absf(y, c[1], 1);
        z = absf(z, c[2], 2);
      }
      if (out.x) out.x[o] = x;
      out.y[o] = y;
      out.z[o] = z;
      out.ux[o] = in.ux[s];
      out.uy[o] = in.uy[s];
      out.uz[o] = in.uz[s];
      out.qw[o] = in.qw[s];
      out.sp[o] = in.sp[s];
      if (out.id) out.id[o] = in.id ? in.id[s] : 0;
      if (keyout) keyout[o] = k;
    }
    if (nt > n) {  // the row's records, in row order: lane = record index
      constexpr int XW = D3 ? PSC_XW3 : PSC_XW2, ND = D3 ? 27 : 9;
      const unsigned mine = lane < ND ? xin.mask[(size_t)k * XW + lane] : 0u;
      int dc = -1;
      for (int d = 0; d < ND; d++)
        if ((__shfl_sync(0xffffffffu, mine, d) >> lane) & 1u) dc = d;
      const bool have = dc >= 0;
      const unsigned m = __ballot_sync(0xffffffffu, have);
      if (have) {
        const size_t idx = (size_t)k * PSC_XCAP + lane, o = (size_t)d0 + n + __popc(m & lanemask_lt());
        const XRec r = xin.rec[idx];
        int sx, sy, sz;
        dir_decode<D3>(dc, sx, sy, sz);
        const int cx = D3 ? wrap_cell(c[0] + sx, gd.n[0]) : 0, cy = wrap_cell(c[1] + sy, gd.n[1]),
                  cz = wrap_cell(c[2] + sz, gd.n[2]);
        float w[8] = {__uint_as_float(r.a.x), __uint_as_float(r.a.y), __uint_as_float(r.a.z), __uint_as_float(r.a.w),
                      __uint_as_float(r.b.x), __uint_as_float(r.b.y), __uint_as_float(r.b.z), __uint_as_float(r.b.w)};
        float x = D3 ? w[0] : w[7], y = D3 ? w[1] : w[0], z = D3 ? w[2] : w[1];
        if (ABS) {
          if (D3) x = absf(x, cx, 0);
          y = absf(y, cy, 1);
          z = absf(z, cz, 2);
        }
        if (out.x) out.x[o] = x;
        out.y[o] = y;
        out.z[o] = z;
        out.ux[o] = D3 ? w[3] : w[2];
        out.uy[o] = D3 ? w[4] : w[3];
        out.uz[o] = D3 ? w[5] : w[4];
        out.qw[o] = D3 ? w[6] : w[5];
        out.sp[o] = __float_as_int(D3 ? w[7] : w[6]);
        if (out.id) out.id[o] = xin.id ? xin.id[idx] : 0;
        if (keyout) keyout[o] = cell_key(gd, cx, cy, cz);
      }
    }
  }
}

// the spill list follows the cells: dense positions doffs[nkeys] ...; *ntotal := all particles
template <bool D3, bool ABS>
__global__ void __launch_bounds__(SORT_THREADS)
k_gather_spill(GridDesc gd, Spill sp, const int *__restrict__ doffs, Cols out, int *__restrict__ keyout,
               int *__restrict__ ntotal, const uint32_t *__restrict__ cond) {
  PSC_COND_RETURN(cond);
  const int ns = min(*sp.count, sp.cap), d0 = doffs[gd.nkeys];
  if (blockIdx.x == 0 && threadIdx.x == 0) *ntotal = d0 + ns;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < ns; i += gridDim.x * blockDim.x) {
    const XRec r = sp.rec[i];
    const int k = sp.key[i];
    const size_t o = (size_t)d0 + i;
    int c[3];
    key_to_cell(gd, k, c);
    auto absf = [&](float off, int cell, int d) {
      float v = __double2float_rn(((double)cell + (double)off) * (double)gd.dx[d]);
      if (v >= gd.L[d]) v = nextafterf(gd.L[d], 0.f);
      return v;
    };
    float w[8] = {__uint_as_float(r.a.x), __uint_as_float(r.a.y), __uint_as_float(r.a.z), __uint_as_float(r.a.w),
                  __uint_as_float(r.b.x), __uint_as_float(r.b.y), __uint_as_float(r.b.z), __uint_as_float(r.b.w)};
    float x = D3 ? w[0] : w[7], y = D3 ? w[1] : w[0], z = D3 ? w[2] : w[1];
    if (ABS) {
      if (D3) x = absf(x, c[0], 0);
      y = absf(y, c[1], 1);
      z = absf(z, c[2], 2);
    }
    if (out.x) out.x[o] = x;
    out.y[o] = y;
    out.z[o] = z;
    out.ux[o] = D3 ? w[3] : w[2];
    out.uy[o] = D3 ? w[4] : w[3];
    out.uz[o] = D3 ? w[5] : w[4];
    out.qw[o] = D3 ? w[6] : w[5];
    out.sp[o] = __float_as_int(D3 ? w[7] : w[6]);
    if (out.id) out.id[o] = sp.id ? sp.id[i] : 0;
    if (keyout) keyout[o] = k;
  }
}

// after a (re-)layout: every exchange row empty, nothing spilled; records the slots in use
__global__ void __launch_bounds__(SORT_THREADS)
k_store_reset(int nk, int xw, uint32_t *__restrict__ m0, uint32_t *__restrict__ m1, uint8_t *__restrict__ bigcell,
              int ntiles, int32_t *__restrict__ bigflag, const int *__restrict__ base, uint32_t *__restrict__ dw, long long capacity,
              const uint32_t *__restrict__ cond) {
  PSC_COND_RETURN(cond);
  const int m = nk * xw;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < m; i += gridDim.x * blockDim.x) {
    m0[i] = 0u;
    m1[i] = 0u;
    if (i < nk) bigcell[i] = 0;
    if (i < ntiles) bigflag[i] = 0;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    dw[PSC_DW_SLOTS] = (uint32_t)base[nk];
    if ((long long)base[nk] > capacity) atomicOr(&dw[PSC_DW_FLAGS], PSC_F_OVERFLOW);
  }
}

// last launch of a conditional re-layout (grid of one block): clears the condition itself
__global__ void k_relayout_done(uint32_t *__restrict__ dw) {
  if (threadIdx.x == 0 && dw[PSC_DW_SPILL]) {
    dw[PSC_DW_SPILL] = 0;
    dw[PSC_DW_RELAYOUTS]++;
  }
}

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace

// slots per column a store of n particles can need (see cell_capacity)
int64_t psc_store_capacity(const psc_ctx *c, int64_t n) {
  const int64_t nk = c->gd.nkeys;
  const int64_t v = n + n / 8 + (int64_t)(6.0 * sqrt((double)nk * (double)n)) + 56 * nk;
  return (v + 31) / 32 * 32;
}

// a quarter of the particles may be homeless at once before PSC_F_OVERFLOW
static int64_t spill_capacity(int64_t n) { return n / 4 > 8192 ? n / 4 : 8192; }

size_t psc_sort_workspace_bytes(const psc_ctx *c, int64_t n) {
  const size_t nk = (size_t)c->gd.nkeys;
  const size_t nx = nk * PSC_XCAP;
  size_t b = 0;
  b += 3 * align_up((size_t)n * 4 + 4, 256);                  // key, perm, cell_idx
  b += 6 * align_up((nk + 1) * 4, 256);                       // offs_dense, base, cnt, cursor, tot, doffs
  b += 2 * align_up((nk + 1) * 8, 256);                       // pack, packloc
  b += align_up((nk / SCAN_TILE + 3) * 8, 256);               // scan_tmp
  b += align_up(((size_t)n / WARP_SEG_CAP + 16) * 4, 256);    // big_list
  b += align_up((size_t)c->gd.ntiles * 4, 256);               // bigflag
  b += align_up(nk, 256);                                     // bigcell
  b += 2 * (align_up(nx * sizeof(XRec), 256) + align_up(nk * PSC_XW3 * 4, 256) + align_up(nx * 4, 256));  // exchange x2
  const size_t sc = (size_t)spill_capacity(n);
  b += align_up(sc * sizeof(XRec), 256) + 2 * align_up(sc * 4, 256);  // spill
  return b;
}

int psc_sort_carve(psc_ctx *c, int64_t n) {
  const size_t nk = (size_t)c->gd.nkeys;
  const size_t nx = nk * PSC_XCAP;
  char *p = (char *)c->ws;
  auto take = [&](size_t bytes) {
    void *r = p;
    p += align_up(bytes, 256);
    return r;
  };
  c->key = (int32_t *)take((size_t)n * 4 + 4);
  c->perm = (int32_t *)take((size_t)n * 4 + 4);
  c->cell_idx = (int32_t *)take((size_t)n * 4 + 4);
  c->offs_dense = (int32_t *)take((nk + 1) * 4);
  c->base = (int32_t *)take((nk + 1) * 4);
  c->cnt = (int32_t *)take((nk + 1) * 4);
  c->cursor = (int32_t *)take((nk + 1) * 4);
  c->tot = (int32_t *)take((nk + 1) * 4);
  c->doffs = (int32_t *)take((nk + 1) * 4);
  c->pack = (long long *)take((nk + 1) * 8);
  c->packloc = (long long *)take((nk + 1) * 8);
  c->scan_tmp = (long long *)take((nk / SCAN_TILE + 3) * 8);
  c->big_list = (int32_t *)take(((size_t)n / WARP_SEG_CAP + 16) * 4);
  c->bigflag = (int32_t *)take((size_t)c->gd.ntiles * 4);
  c->bigcell = (uint8_t *)take(nk);
  for (int i = 0; i < 2; i++) {
    c->xch[i].rec = (XRec *)take(nx * sizeof(XRec));
    c->xch[i].mask = (uint32_t *)take(nk * PSC_XW3 * 4);
    c->xch[i].id = (int32_t *)take(nx * 4);
  }
  const size_t sc = (size_t)spill_capacity(n);
  c->spill.rec = (XRec *)take(sc * sizeof(XRec));
  c->spill.key = (int32_t *)take(sc * 4);
  c->spill.id = (int32_t *)take(sc * 4);
  c->spill.count = (int32_t *)(c->d_flags + PSC_DW_SPILL);
  c->spill.cap = (int)sc;
  if ((size_t)(p - (char *)c->ws) > c->ws_bytes) return PSC_ERR_WORKSPACE;
  return PSC_OK;
}

// what the particle kernels see: the current column set in buffer-column order, the exchange
// the last push filled (xin) and the one the next push fills (xout)
StoreDesc psc_store_desc(const psc_ctx *c) {
  StoreDesc sd;
  const Cols &p = c->cols[c->cur];
  const bool d3 = psc_is3d(c->gd);
  for (int i = 0; i < 10; i++) sd.col[i] = nullptr;
  int k = 0;
  if (d3) sd.col[k++] = p.x;
  sd.col[k++] = p.y;
  sd.col[k++] = p.z;
  sd.col[k++] = p.ux;
  sd.col[k++] = p.uy;
  sd.col[k++] = p.uz;
  sd.ndyn = k;
  sd.col[k++] = p.qw;
  sd.col[k++] = (float *)p.sp;
  sd.icol_x2d = sd.icol_id = -1;
  if (!d3 && p.x) { sd.icol_x2d = k; sd.col[k++] = p.x; }
  if (p.id) { sd.icol_id = k; sd.col[k++] = (float *)p.id; }
  sd.ncol = k;
  sd.base = c->base;
  sd.cnt = c->cnt;
  sd.xin = c->xch[c->xcur];
  sd.xout = c->xch[c->xcur ^ 1];
  if (!p.id) sd.xin.id = sd.xout.id = nullptr;
  sd.spill = c->spill;
  if (!p.id) sd.spill.id = nullptr;
  sd.imgC = c->bufC;
  sd.bigflag = c->bigflag;
  sd.bigcell = c->bigcell;
  sd.nbig = c->d_flags + PSC_DW_NBIG + c->xcur;
  sd.nbig_next = c->d_flags + PSC_DW_NBIG + (c->xcur ^ 1);
  sd.flags = c->d_flags + PSC_DW_FLAGS;
  sd.maxcnt = c->d_flags + PSC_DW_MAXCNT;
  sd.maxcnt_known = c->maxcnt_known;
  return sd;
}

namespace {

// packed scan of c->pack -> base (capacities), offs_dense (counts), cursor := offs_dense
int run_scan2(psc_ctx *c, cudaStream_t s, const uint32_t *cond) {
  const int nk = c->gd.nkeys;
  ProfScope ps(c, PSC_PH_SORT_SCAN, s);
  const int sblocks = (int)cdiv64(nk, SCAN_TILE);
  k_scan_local<long long><<<sblocks, SORT_THREADS, 0, s>>>(nk, c->pack, c->packloc, c->scan_tmp, cond);
  PSC_LAUNCH_CHECK(c);
  k_scan_tmp<long long><<<1, 1024, 0, s>>>(sblocks, c->scan_tmp, cond);
  PSC_LAUNCH_CHECK(c);
  k_scan_add2<<<sblocks, SORT_THREADS, 0, s>>>(nk, c->packloc, c->base, c->offs_dense, c->cursor,
                                               c->scan_tmp, sblocks, cond);
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}

// exclusive scan tot -> doffs
int run_scan1(psc_ctx *c, cudaStream_t s, const uint32_t *cond) {
  const int nk = c->gd.nkeys;
  const int sblocks = (int)cdiv64(nk, SCAN_TILE);
  int *tmp = (int *)c->scan_tmp;
  k_scan_local<int><<<sblocks, SORT_THREADS, 0, s>>>(nk, c->tot, c->doffs, tmp, cond);
  PSC_LAUNCH_CHECK(c);
  k_scan_tmp<int><<<1, 1024, 0, s>>>(sblocks, tmp, cond);
  PSC_LAUNCH_CHECK(c);
  k_scan_add<<<sblocks, SORT_THREADS, 0, s>>>(nk, c->doffs, nullptr, tmp, sblocks, cond);
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}

int grid_for(const psc_ctx *c, int64_t items, int per_block) {
  return (int)min((int64_t)c->sm_count * 16, max((int64_t)1, cdiv64(items, per_block)));
}

// flattens the store of the current set into `dst` (dense), keys into keyout; *ntotal (device)
// receives the particle count
int gather_store(psc_ctx *c, const Cols &dst, int32_t *keyout, bool to_abs, int *ntotal, cudaStream_t s,
                 const uint32_t *cond) {
  const GridDesc &gd = c->gd;
  const int nk = gd.nkeys;
  const Cols &in = c->cols[c->cur];
  const Exchange &xin = c->xch[c->xcur];
  Exchange xi = xin;
  Spill sp = c->spill;
  if (!in.id) { xi.id = nullptr; sp.id = nullptr; }
  k_tot<<<grid_for(c, nk, SORT_THREADS), SORT_THREADS, 0, s>>>(nk, psc_is3d(gd) ? PSC_XW3 : PSC_XW2, gd.nd, c->cnt,
                                                              xin.mask, c->tot, cond);
  PSC_LAUNCH_CHECK(c);
  int rc = run_scan1(c, s, cond);
  if (rc) return rc;
  const int gb = grid_for(c, nk, SORT_THREADS / 32);
  const int sb = grid_for(c, c->spill.cap, SORT_THREADS);
  const bool d3 = psc_is3d(gd);
#define PSC_GATHER(D3_, ABS_)                                                                        \
  do {                                                                                               \
    k_gather<D3_, ABS_><<<gb, SORT_THREADS, 0, s>>>(gd, in, c->base, c->cnt, xi, c->doffs, dst, keyout, cond); \
    PSC_LAUNCH_CHECK(c);                                                                             \
    k_gather_spill<D3_, ABS_><<<sb, SORT_THREADS, 0, s>>>(gd, sp, c->doffs, dst, keyout, ntotal, cond);       \
    PSC_LAUNCH_CHECK(c);                                                                             \
  } while (0)
  if (d3 && to_abs) PSC_GATHER(true, true);
  else if (d3) PSC_GATHER(true, false);
  else if (to_abs) PSC_GATHER(false, true);
  else PSC_GATHER(false, false);
#undef PSC_GATHER
  return PSC_OK;
}

// counting sort of the dense list `src` (keys in c->key, histogram in c->cursor, *np particles)
// into the store layout in `dst`
int sort_core(psc_ctx *c, const Cols &src, const Cols &dst, bool from_abs, bool stable, const int *np,
              cudaStream_t s, const uint32_t *cond) {
  const GridDesc &gd = c->gd;
  const int nk = gd.nkeys;
  const int pblocks = grid_for(c, c->np, SORT_THREADS);
  k_layout<<<grid_for(c, nk, SORT_THREADS), SORT_THREADS, 0, s>>>(nk, c->cursor, c->pack, c->cnt, c->d_flags, cond);
  PSC_LAUNCH_CHECK(c);
  int rc = run_scan2(c, s, cond);
  if (rc) return rc;
  psc_prof_begin(c, PSC_PH_SORT_RANK, s);
  k_scatter<<<pblocks, SORT_THREADS, 0, s>>>(np, c->key, c->cursor, c->perm, cond);
  PSC_LAUNCH_CHECK(c);
  if (stable) {
    const int kblocks = (int)min((int64_t)c->sm_count * 64, max((int64_t)1, cdiv64(nk, SORT_THREADS / 32)));
    k_segsort<<<kblocks, SORT_THREADS, 0, s>>>(nk, c->offs_dense, c->perm, c->big_list, c->d_flags + PSC_DW_BIG);
    PSC_LAUNCH_CHECK(c);
    if (c->np > WARP_SEG_CAP) {
      static bool attr_set = false;
      if (!attr_set) {
        PSC_CUDA_TRY(c, cudaFuncSetAttribute(k_segsort_big, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             BIG_SMEM_CAP * 4));
        attr_set = true;
      }
      k_segsort_big<<<c->sm_count, 1024, BIG_SMEM_CAP * 4, s>>>(c->offs_dense, c->perm, c->big_list,
                                                                c->d_flags + PSC_DW_BIG);
      PSC_LAUNCH_CHECK(c);
    }
  }
  psc_prof_end(c, PSC_PH_SORT_RANK, s);
  psc_prof_begin(c, PSC_PH_SORT_REORDER, s);
  if (from_abs)
    k_reorder<true><<<pblocks, SORT_THREADS, 0, s>>>(gd, np, c->perm, c->key, c->offs_dense, c->base, src, dst, cond);
  else
    k_reorder<false><<<pblocks, SORT_THREADS, 0, s>>>(gd, np, c->perm, c->key, c->offs_dense, c->base, src, dst, cond);
  PSC_LAUNCH_CHECK(c);
  psc_prof_end(c, PSC_PH_SORT_REORDER, s);
  k_store_reset<<<grid_for(c, (int64_t)nk * 16, SORT_THREADS), SORT_THREADS, 0, s>>>(
      nk, psc_is3d(gd) ? PSC_XW3 : PSC_XW2, c->xch[0].mask, c->xch[1].mask, c->bigcell, gd.ntiles, c->bigflag,
      c->base, c->d_flags,
      (long long)c->capacity, cond);
  PSC_LAUNCH_CHECK(c);
  return PSC_OK;
}

}  // namespace

int psc_store_gather(psc_ctx *c, const Cols &dst, int32_t *key, bool to_abs, cudaStream_t s) {
  return gather_store(c, dst, key, to_abs, c->key + c->np /* scratch word behind key[] */, s, nullptr);
}

// Size of the per-warp cell image of the particle kernels: the largest cell of the last layout
// plus room for its arrivals.  Called whenever the host has the status block anyway (after the
// general sort, in psc_status / psc_store_info): a device-side re-layout of a run that clumps
// raises the largest count, and the image follows at the next such call (it never shrinks).
void psc_refresh_image_size(psc_ctx *c, const uint32_t *dw) {
  const int mx = (int)dw[PSC_DW_MAXCNT];
  c->maxcnt_known = mx;
  int C = (mx + mx / 8 + 24 + 31) / 32 * 32;  // 64, 96, ..., 256
  C = C < 64 ? 64 : (C > 256 ? 256 : C);
  // the order-2 kernel is bound by registers (2 blocks/SM), not by shared memory: it takes the largest
  // image, so that cells which fill up while a run clumps stay on the image path
  if (c->gd.order == 2) C = 256;
  if (C > c->bufC) c->bufC = C;
}

// general counting sort: any state in, the cell store (stable inside every cell) out
int psc_sort_general(psc_ctx *c, cudaStream_t s) {
  const GridDesc &gd = c->gd;
  const int n = (int)c->np;
  const int nk = gd.nkeys;
  const int pblocks = grid_for(c, n, SORT_THREADS);
  int *np_dev = c->key + c->np;  // one scratch word behind key[]: the particle count on the device
  PSC_CUDA_TRY(c, cudaMemsetAsync(c->cursor, 0, (size_t)(nk + 1) * 4, s));
  PSC_CUDA_TRY(c, cudaMemsetAsync(c->d_flags + PSC_DW_BIG, 0, 4, s));
  PSC_CUDA_TRY(c, cudaMemsetAsync(c->d_flags + PSC_DW_MAXCNT, 0, 4, s));
  c->launches += 3;
  const bool from_abs = c->form == PSC_FORM_ABS;
  const Cols &src = c->cols[from_abs ? c->cur : c->cur ^ 1];
  const Cols &dst = c->cols[from_abs ? c->cur ^ 1 : c->cur];
  psc_prof_begin(c, PSC_PH_SORT_COUNT, s);
  if (from_abs) {
    c->np32 = n;
    PSC_CUDA_TRY(c, cudaMemcpyAsync(np_dev, &c->np32, 4, cudaMemcpyHostToDevice, s));
    k_keys<<<pblocks, SORT_THREADS, 0, s>>>(gd, n, src.x, src.y, src.z, src.sp, c->key, c->cursor,
                                            c->d_flags + PSC_DW_FLAGS);
    PSC_LAUNCH_CHECK(c);
  } else {  // a store sorted again: flatten it into the other set, keys from the cells
    const int rc = gather_store(c, src, c->key, false, np_dev, s, nullptr);
    if (rc) return rc;
    k_hist<<<pblocks, SORT_THREADS, 0, s>>>(np_dev, nk, c->key, c->cursor, c->d_flags + PSC_DW_FLAGS, nullptr);
    PSC_LAUNCH_CHECK(c);
  }
  psc_prof_end(c, PSC_PH_SORT_COUNT, s);
  {
    const int rc = sort_core(c, src, dst, from_abs, true, np_dev, s, nullptr);
    if (rc) return rc;
  }
  PSC_CUDA_TRY(c, cudaMemsetAsync(c->d_flags + PSC_DW_SPILL, 0, 4, s));
  if (from_abs) c->cur ^= 1;
  c->xcur = 0;
  c->form = PSC_FORM_REL;
  c->state = PSC_STATE_STORE;
  c->have_sort_result = 1;
  // size of the per-warp cell image of the particle kernels: the largest cell plus room for its
  // arrivals (read back: this call synchronises the stream)
  uint32_t dw[PSC_DW_COUNT];
  PSC_CUDA_TRY(c, cudaMemcpyAsync(dw, c->d_flags, sizeof(dw), cudaMemcpyDeviceToHost, s));
  PSC_CUDA_TRY(c, cudaStreamSynchronize(s));
  c->bufC = 0;
  psc_refresh_image_size(c, dw);
  if ((int64_t)dw[PSC_DW_SLOTS] > c->capacity) return PSC_ERR_WORKSPACE;
  return PSC_OK;
}

// in the steady state nothing is sorted.  Only if the last push spilled
// (device word PSC_DW_SPILL != 0) the store is flattened and laid out again.  Whether that is
// needed is known on the device only, so the step launches ONE single-thread kernel that looks at
// the word and, if it is set, launches the chain itself (CUDA dynamic parallelism, tail launches:
// they run in order after the launcher and before the next kernel of the stream).
namespace {

struct RelayoutArgs {
  GridDesc gd;
  Cols cur, tmp;         // the store's column set; the other one (dense scratch)
  Exchange xin, x0, x1;  // the exchange holding the last push's records; both, for the reset
  Spill spill;
  int32_t *key, *perm, *offs_dense, *base, *cnt, *cursor, *tot, *doffs;
  uint8_t *bigcell;
  int32_t *bigflag;
  long long *pack, *packloc, *scan_tmp;
  uint32_t *dw;
  int *np_dev;
  long long capacity;
  int g_cells, g_warpcells, g_part, g_spill, g_reset, sblocks;
};

template <bool D3>
__device__ void relayout_chain(const RelayoutArgs &a) {
  const int nk = a.gd.nkeys, T = SORT_THREADS;
  const cudaStream_t ts = cudaStreamTailLaunch;
  const uint32_t *nc = nullptr;
  constexpr int XW = D3 ? PSC_XW3 : PSC_XW2;
  // flatten: residents + exchange records + spill list -> tmp (dense), keys -> key
  k_tot<<<a.g_cells, T, 0, ts>>>(nk, XW, a.gd.nd, a.cnt, a.xin.mask, a.tot, nc);
  k_scan_local<int><<<a.sblocks, T, 0, ts>>>(nk, a.tot, a.doffs, (int *)a.scan_tmp, nc);
  k_scan_tmp<int><<<1, 1024, 0, ts>>>(a.sblocks, (int *)a.scan_tmp, nc);
  k_scan_add<<<a.sblocks, T, 0, ts>>>(nk, a.doffs, nullptr, (const int *)a.scan_tmp, a.sblocks, nc);
  k_gather<D3, false><<<a.g_warpcells, T, 0, ts>>>(a.gd, a.cur, a.base, a.cnt, a.xin, a.doffs, a.tmp, a.key, nc);
  k_gather_spill<D3, false><<<a.g_spill, T, 0, ts>>>(a.gd, a.spill, a.doffs, a.tmp, a.key, a.np_dev, nc);
  // count, lay out, scatter back
  k_zero<<<a.g_cells, T, 0, ts>>>(nk + 1, a.cursor, nc);
  k_hist<<<a.g_part, T, 0, ts>>>(a.np_dev, nk, a.key, a.cursor, a.dw + PSC_DW_FLAGS, nc);
  k_layout<<<a.g_cells, T, 0, ts>>>(nk, a.cursor, a.pack, a.cnt, a.dw, nc);
  k_scan_local<long long><<<a.sblocks, T, 0, ts>>>(nk, a.pack, a.packloc, a.scan_tmp, nc);
  k_scan_tmp<long long><<<1, 1024, 0, ts>>>(a.sblocks, a.scan_tmp, nc);
  k_scan_add2<<<a.sblocks, T, 0, ts>>>(nk, a.packloc, a.base, a.offs_dense, a.cursor, a.scan_tmp, a.sblocks, nc);
  k_scatter<<<a.g_part, T, 0, ts>>>(a.np_dev, a.key, a.cursor, a.perm, nc);
  k_reorder<false><<<a.g_part, T, 0, ts>>>(a.gd, a.np_dev, a.perm, a.key, a.offs_dense, a.base, a.tmp, a.cur, nc);
  k_store_reset<<<a.g_reset, T, 0, ts>>>(nk, XW, a.x0.mask, a.x1.mask, a.bigcell, a.gd.ntiles, a.bigflag, a.base,
                                         a.dw, a.capacity, nc);
  k_relayout_done<<<1, 32, 0, ts>>>(a.dw);
}

// A spilled particle (the 33rd leaver of a cell in one step, mostly) does not need a re-layout if
// its destination cell has a free slot: one block files the spill list straight into the cells
// and keeps, compacted at the front of the list, only those that found no room.
constexpr int SPILL_INSERT_MAX = 1 << 16;  // longer lists (mass migration) go to the re-layout at once
template <bool D3>
__global__ void __launch_bounds__(256) k_spill_insert(RelayoutArgs a) {
  __shared__ int nfail;
  const int ns = min(*a.spill.count, a.spill.cap);
  if (threadIdx.x == 0) nfail = 0;
  __syncthreads();
  for (int i0 = 0; i0 < ns; i0 += blockDim.x) {
    const int i = i0 + threadIdx.x;
    const bool have = i < ns;
    XRec r;
    int key = 0, id = 0;
    r.a = r.b = make_uint4(0, 0, 0, 0);
    if (have) {
      r = a.spill.rec[i];
      key = a.spill.key[i];
      if (a.spill.id) id = a.spill.id[i];
    }
    __syncthreads();  // the whole chunk is read before anything is written over the list's front
    bool fail = false;
    if (have) {
      const int slot = atomicAdd(&a.cnt[key], 1);
      if (slot < a.base[key + 1] - a.base[key]) {
        const size_t o = (size_t)a.base[key] + slot;
        const float w[8] = {__uint_as_float(r.a.x), __uint_as_float(r.a.y), __uint_as_float(r.a.z),
                            __uint_as_float(r.a.w), __uint_as_float(r.b.x), __uint_as_float(r.b.y),
                            __uint_as_float(r.b.z), __uint_as_float(r.b.w)};
        if (D3) a.cur.x[o] = w[0];
        else if (a.cur.x) a.cur.x[o] = w[7];
        a.cur.y[o] = D3 ? w[1] : w[0];
        a.cur.z[o] = D3 ? w[2] : w[1];
        a.cur.ux[o] = D3 ? w[3] : w[2];
        a.cur.uy[o] = D3 ? w[4] : w[3];
        a.cur.uz[o] = D3 ? w[5] : w[4];
        a.cur.qw[o] = D3 ? w[6] : w[5];
        a.cur.sp[o] = __float_as_int(D3 ? w[7] : w[6]);
        if (a.cur.id) a.cur.id[o] = id;
        atomicMax(&a.dw[PSC_DW_MAXCNT], (uint32_t)(slot + 1));
      } else {
        atomicSub(&a.cnt[key], 1);
        fail = true;
      }
    }
    if (fail) {
      const int f = atomicAdd(&nfail, 1);
      a.spill.rec[f] = r;
      a.spill.key[f] = key;
      if (a.spill.id) a.spill.id[f] = id;
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    a.dw[PSC_DW_INSERTED] += (uint32_t)(ns - nfail);
    *a.spill.count = nfail;
  }
}

// second look at the spill counter, after the insertion: what is left needs the re-layout
__global__ void k_relayout_gate2(RelayoutArgs a) {
  if (threadIdx.x != 0 || a.dw[PSC_DW_SPILL] == 0) return;
  if (a.gd.n[0] > 1) relayout_chain<true>(a);
  else relayout_chain<false>(a);
}

__global__ void k_relayout_gate(RelayoutArgs a) {
  if (threadIdx.x != 0) return;
  const uint32_t ns = a.dw[PSC_DW_SPILL];
  if (ns == 0) return;
  if (ns <= (uint32_t)SPILL_INSERT_MAX && ns <= (uint32_t)a.spill.cap) {
    if (a.gd.n[0] > 1) k_spill_insert<true><<<1, 256, 0, cudaStreamTailLaunch>>>(a);
    else k_spill_insert<false><<<1, 256, 0, cudaStreamTailLaunch>>>(a);
    k_relayout_gate2<<<1, 32, 0, cudaStreamTailLaunch>>>(a);
  } else if (a.gd.n[0] > 1) {
    relayout_chain<true>(a);
  } else {
    relayout_chain<false>(a);
  }
}

}  // namespace

int psc_store_relayout_if_spilled(psc_ctx *c, cudaStream_t s) {
  const int nk = c->gd.nkeys;
  RelayoutArgs a;
  a.gd = c->gd;
  a.cur = c->cols[c->cur];
  a.tmp = c->cols[c->cur ^ 1];
  a.xin = c->xch[c->xcur];
  a.x0 = c->xch[0];
  a.x1 = c->xch[1];
  a.spill = c->spill;
  if (!a.cur.id) {
    a.xin.id = nullptr;
    a.spill.id = nullptr;
  }
  a.key = c->key; a.perm = c->perm; a.offs_dense = c->offs_dense; a.base = c->base; a.cnt = c->cnt;
  a.cursor = c->cursor; a.tot = c->tot; a.doffs = c->doffs; a.bigcell = c->bigcell;
  a.bigflag = c->bigflag;
  a.pack = c->pack; a.packloc = c->packloc; a.scan_tmp = c->scan_tmp;
  a.dw = c->d_flags;
  a.np_dev = c->key + c->np;
  a.capacity = (long long)c->capacity;
  a.g_cells = grid_for(c, nk, SORT_THREADS);
  a.g_warpcells = grid_for(c, nk, SORT_THREADS / 32);
  a.g_part = grid_for(c, c->np, SORT_THREADS);
  a.g_spill = grid_for(c, c->spill.cap, SORT_THREADS);
  a.g_reset = grid_for(c, (int64_t)nk * 16, SORT_THREADS);
  a.sblocks = (int)cdiv64(nk, SCAN_TILE);
  k_relayout_gate<<<1, 32, 0, s>>>(a);
  PSC_LAUNCH_CHECK(c);
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
