// Device-side neighbour list (the paper's rates are atom-timesteps/s with the list
// build inside; the GPU runs use the host code's list): the full CSR list mtp_compute consumes, its
// image shifts and its reverse index, built from positions and box with a cell list, and the two halves of a
// velocity-Verlet step.  Integer work: the result is bit-identical to a brute-force search over the 27 images
// (rows ordered by (j, shift), the order of oracle/mtp.py brute_force_neighbours; tests compare bit for bit).
//
//   cells    the box is cut into n_k = floor(height_k / r_list) >= 1 cells per lattice direction (fractional
//            coordinates), so a neighbour image lies in one of the 27 cells around the centre atom's; the image shift of
//            a candidate is the number of box lengths the cell index wrapped by.  With fewer than three cells in a
//            direction the same cell is visited through different shifts -- still every image in {-1,0,1}^3 exactly once.
//   build    cell index per atom + histogram -> exclusive scan -> atoms sorted by cell (each cell's atoms in ascending
//            order) with a cell-ordered copy of the wrapped positions -> per atom (one warp): count pass -> scan ->
//            fill pass: hits collected in shared memory, rank-sorted by key j * 27 + code, written as idx / shift.
//   rev      per pair a binary search of the mirror key (i, -s) in row j.
// The distance test uses the same operation order as the definition, (x_j - x_i) + s0 H0 + s1 H1 + s2 H2, without
// contractions, on the caller's coordinates.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include "kernels.h"
#include "mtp_b200.h"

namespace mtpb {

namespace {
constexpr int kRowMax = 256;            // longest row the fill pass sorts in shared memory (longer rows: flag[0] counts them)

__device__ __forceinline__ int cell_of(const NbGrid &g, double x, double y, double z, int *w) {
  // fractional coordinates (row-vector convention frac = cart . Hi), wrapped into [0, 1)
  double f0 = x * g.Hi[0] + y * g.Hi[3] + z * g.Hi[6];
  double f1 = x * g.Hi[1] + y * g.Hi[4] + z * g.Hi[7];
  double f2 = x * g.Hi[2] + y * g.Hi[5] + z * g.Hi[8];
  const double w0 = floor(f0), w1 = floor(f1), w2 = floor(f2);
  f0 -= w0; f1 -= w1; f2 -= w2;
  w[0] = (int)w0; w[1] = (int)w1; w[2] = (int)w2;
  const int c0 = min((int)(f0 * g.nc[0]), g.nc[0] - 1), c1 = min((int)(f1 * g.nc[1]), g.nc[1] - 1), c2 = min((int)(f2 * g.nc[2]), g.nc[2] - 1);
  return (c0 * g.nc[1] + c1) * g.nc[2] + c2;
}

// cell index and wrap image of every atom; histogram of the cells
__global__ void k_nb_cells(NbGrid g, const double *__restrict__ pos, int n, int *__restrict__ cell, int *__restrict__ wrap,
                           int *__restrict__ count, int *__restrict__ flag) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int w[3];
  const double x = pos[3 * (size_t)i], y = pos[3 * (size_t)i + 1], z = pos[3 * (size_t)i + 2];
  int c = 0;
  // a coordinate that is not finite, or further out than 2^30 box lengths (an MD run that blew up): counted as an
  // error, the atom goes to cell 0 and gets no neighbours (its distance tests fail)
  const double big = 1073741824.0;
  const double f0 = x * g.Hi[0] + y * g.Hi[3] + z * g.Hi[6], f1 = x * g.Hi[1] + y * g.Hi[4] + z * g.Hi[7], f2 = x * g.Hi[2] + y * g.Hi[5] + z * g.Hi[8];
  if (fabs(f0) < big && fabs(f1) < big && fabs(f2) < big) c = cell_of(g, x, y, z, w);
  else { w[0] = w[1] = w[2] = 0; atomicAdd(flag, 1); }
  cell[i] = c;
  wrap[3 * (size_t)i] = w[0]; wrap[3 * (size_t)i + 1] = w[1]; wrap[3 * (size_t)i + 2] = w[2];
  atomicAdd(count + c, 1);
}

// ---- exclusive scan of int32 counts into int64 offsets: blocks of 1024, block totals scanned by a second level
__global__ void __launch_bounds__(1024) k_scan_block(const int *__restrict__ in, long long n, long long *__restrict__ out,
                                                     long long *__restrict__ totals) {
  __shared__ long long sm[1024];
  const long long i = (long long)blockIdx.x * 1024 + threadIdx.x;
  const long long v = i < n ? in[i] : 0;
  sm[threadIdx.x] = v;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    const long long t = threadIdx.x >= o ? sm[threadIdx.x - o] : 0;
    __syncthreads();
    sm[threadIdx.x] += t;
    __syncthreads();
  }
  if (i < n) out[i] = sm[threadIdx.x] - v;
  if (threadIdx.x == 1023) totals[blockIdx.x] = sm[1023];
}
__global__ void __launch_bounds__(1024) k_scan_totals(long long *__restrict__ totals, int nblocks, long long *__restrict__ grand) {
  // one block: exclusive scan of up to 1024 * 1024 block totals, 1024 at a time with a running carry
  __shared__ long long sm[1024];
  __shared__ long long carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int base = 0; base < nblocks; base += 1024) {
    const int i = base + threadIdx.x;
    const long long v = i < nblocks ? totals[i] : 0;
    sm[threadIdx.x] = v;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
      const long long t = threadIdx.x >= o ? sm[threadIdx.x - o] : 0;
      __syncthreads();
      sm[threadIdx.x] += t;
      __syncthreads();
    }
    if (i < nblocks) totals[i] = carry + sm[threadIdx.x] - v;
    __syncthreads();
    if (threadIdx.x == 1023) carry += sm[1023];
    __syncthreads();
  }
  if (threadIdx.x == 0) *grand = carry;
}
__global__ void __launch_bounds__(1024) k_scan_add(long long *__restrict__ out, long long n, const long long *__restrict__ totals,
                                                   const long long *__restrict__ grand) {
  const long long i = (long long)blockIdx.x * 1024 + threadIdx.x;
  if (i < n) out[i] += totals[blockIdx.x];
  if (i == n) out[n] = *grand;            // the closing offset
}
}  // namespace

// out[0 .. n] = exclusive prefix sums of in[0 .. n) (out[n] = total); totals: scratch of ceil(n / 1024) + 1 int64
cudaError_t launch_scan(const int *in, long long n, long long *out, long long *totals, cudaStream_t st) {
  const int nblocks = (int)((n + 1 + 1023) / 1024);      // + 1: some block must own index n for the closing offset
  k_scan_block<<<nblocks, 1024, 0, st>>>(in, n, out, totals);
  k_scan_totals<<<1, 1024, 0, st>>>(totals, nblocks, totals + nblocks);
  k_scan_add<<<nblocks, 1024, 0, st>>>(out, n, totals, totals + nblocks);
  count_launch(); count_launch(); count_launch();
  return cudaGetLastError();
}


namespace {
// atoms into their cells (any order), then each cell's atoms in ascending order: the candidate order is deterministic
__global__ void k_nb_scatter(const int *__restrict__ cell, int n, const long long *__restrict__ start, int *__restrict__ cursor,
                             int *__restrict__ sorted) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int c = cell[i];
  sorted[start[c] + atomicAdd(cursor + c, 1)] = i;
}
__global__ void k_nb_sort_cells(const long long *__restrict__ start, int n_cells, int *__restrict__ sorted) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_cells) return;
  const long long a = start[c], b = start[c + 1];
  for (long long p = a + 1; p < b; ++p) {            // insertion sort: a cell holds about ten atoms
    const int v = sorted[p];
    long long q = p;
    while (q > a && sorted[q - 1] > v) { sorted[q] = sorted[q - 1]; --q; }
    sorted[q] = v;
  }
}
// the caller's coordinates of the atoms in cell order: one 32-byte record (x, y, z, tag) per candidate, tag = atom
// index, + 2^27 when the atom lies outside the box (its wrap image is then read from wrap[]; the common case needs no
// second load)
constexpr int kWrapBit = 1 << 27;
__global__ void k_nb_gather_pos(const double *__restrict__ pos, const int *__restrict__ sorted, const int *__restrict__ wrap, int n,
                                double *__restrict__ pos_s) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  const int i = sorted[t];
  const bool out = (wrap[3 * (size_t)i] | wrap[3 * (size_t)i + 1] | wrap[3 * (size_t)i + 2]) != 0;
  double2 *o = reinterpret_cast<double2 *>(pos_s) + 2 * (size_t)t;
  o[0] = make_double2(pos[3 * (size_t)i], pos[3 * (size_t)i + 1]);
  o[1] = make_double2(pos[3 * (size_t)i + 2], (double)(i + (out ? kWrapBit : 0)));
}

// One warp per atom (in cell order).  The 27 cells around its cell are 27 segments of the cell-sorted records; lane
// d < 27 looks up segment d (begin, size, image of the cell wrap), a warp scan lays the segments end to end, and the
// lanes then walk the concatenated candidates 32 at a time -- full lanes whatever the cell occupancy.
// MODE 0 (count): count[i] = number of neighbours.
// MODE 1 (fill):  the row's keys j * 27 + code are collected in shared memory, rank-sorted, and written as idx / shift
//                 at off[i] (coalesced).  if_truncated: only when off[n] > capacity (see MODE 2).
// MODE 2 (stash): one search instead of two: count[i] as MODE 0, and the sorted keys of the row go to tmp at a place
//                 claimed from a global cursor (tstart[i]; -1 when it lies beyond the capacity); k_nb_place moves them
//                 to off[i] once the offsets are known.  When the list does not fit its capacity the stash is
//                 incomplete: k_nb_place then does nothing and a MODE 1 pass writes the first `capacity` pairs.
enum { NB_COUNT = 0, NB_FILL = 1, NB_STASH = 2 };
template <int MODE>
__global__ void __launch_bounds__(256) k_nb_rows(NbGrid g, const double *__restrict__ pos_s, const int *__restrict__ cell,
                                                 const int *__restrict__ wrap, const long long *__restrict__ start, int n, double r2max,
                                                 int *__restrict__ count, const long long *__restrict__ off, long long capacity,
                                                 int *__restrict__ idx, signed char *__restrict__ shift, int *__restrict__ flag,
                                                 int if_truncated, int *__restrict__ tstart, unsigned *__restrict__ tmp,
                                                 unsigned long long *__restrict__ cursor) {
  constexpr bool FILL = MODE != NB_COUNT;
  __shared__ unsigned keys[FILL ? 8 : 1][FILL ? kRowMax : 1], sorted_keys[FILL ? 8 : 1][FILL ? kRowMax : 1];
  if (MODE == NB_FILL && if_truncated && off[n] <= capacity) return;
  __shared__ long long seg_base[8][27];
  __shared__ int seg_end[8][27], seg_m[8][27];
  const unsigned full = 0xffffffffu;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int t = blockIdx.x * 8 + wib;                       // position in cell order
  if (t >= n) return;
  const double2 a0 = reinterpret_cast<const double2 *>(pos_s)[2 * (size_t)t], a1 = reinterpret_cast<const double2 *>(pos_s)[2 * (size_t)t + 1];
  const int tag_i = (int)a1.y, i = tag_i & (kWrapBit - 1);
  const double xi = a0.x, yi = a0.y, zi = a1.x;
  const int ci = cell[i];
  const int c2 = ci % g.nc[2], c1 = (ci / g.nc[2]) % g.nc[1], c0 = ci / (g.nc[2] * g.nc[1]);
  int wi0 = 0, wi1 = 0, wi2 = 0;
  if (tag_i & kWrapBit) { wi0 = wrap[3 * (size_t)i]; wi1 = wrap[3 * (size_t)i + 1]; wi2 = wrap[3 * (size_t)i + 2]; }
  {
    long long a = 0;
    int size = 0, mcode = 0;
    if (lane < 27) {
      // neighbour cell, wrapped into the grid; the number of box lengths it wrapped by is the image of the wrapped
      // coordinates.  e is in [-1, nc], so one conditional step does it (with nc < 3 the same cell comes up through
      // different images -- still every image exactly once)
      int e0 = c0 + lane / 9 - 1, e1 = c1 + (lane / 3) % 3 - 1, e2 = c2 + lane % 3 - 1, m0 = 0, m1 = 0, m2 = 0;
      if (e0 < 0) { e0 += g.nc[0]; m0 = -1; } else if (e0 >= g.nc[0]) { e0 -= g.nc[0]; m0 = 1; }
      if (e1 < 0) { e1 += g.nc[1]; m1 = -1; } else if (e1 >= g.nc[1]) { e1 -= g.nc[1]; m1 = 1; }
      if (e2 < 0) { e2 += g.nc[2]; m2 = -1; } else if (e2 >= g.nc[2]) { e2 -= g.nc[2]; m2 = 1; }
      const int cj = (e0 * g.nc[1] + e1) * g.nc[2] + e2;
      a = start[cj];
      size = (int)(start[cj + 1] - a);
      mcode = (m0 + 1) * 9 + (m1 + 1) * 3 + (m2 + 1);
    }
    int inc = size;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(full, inc, o); if (lane >= o) inc += v; }
    if (lane < 27) { seg_base[wib][lane] = a - (inc - size); seg_end[wib][lane] = inc; seg_m[wib][lane] = mcode; }
  }
  __syncwarp();
  const int total = seg_end[wib][26];
  int n_row = 0, d = 0;
  for (int tt = lane; tt < ((total + 31) & ~31); tt += 32) {          // whole warp iterations (ballots inside)
    bool hit = false;
    unsigned key = 0;
    if (tt < total) {
      while (tt >= seg_end[wib][d]) ++d;
      const long long p = seg_base[wib][d] + tt;
      const int mc = seg_m[wib][d];
      const double2 b0 = reinterpret_cast<const double2 *>(pos_s)[2 * (size_t)p], b1 = reinterpret_cast<const double2 *>(pos_s)[2 * (size_t)p + 1];
      const int tag_j = (int)b1.y, j = tag_j & (kWrapBit - 1);
      // image shift relative to the caller's (possibly unwrapped) coordinates
      int s0 = mc / 9 - 1 + wi0, s1 = (mc / 3) % 3 - 1 + wi1, s2 = mc % 3 - 1 + wi2;
      if (tag_j & kWrapBit) { s0 -= wrap[3 * (size_t)j]; s1 -= wrap[3 * (size_t)j + 1]; s2 -= wrap[3 * (size_t)j + 2]; }
      if (s0 >= -1 && s0 <= 1 && s1 >= -1 && s1 <= 1 && s2 >= -1 && s2 <= 1 && !(j == i && s0 == 0 && s1 == 0 && s2 == 0)) {
        // r = (x_j - x_i) + s0 H0 + s1 H1 + s2 H2, no contractions (the definition's rounding)
        const double x = __dadd_rn(__dadd_rn(__dadd_rn(__dadd_rn(b0.x, -xi), __dmul_rn((double)s0, g.H[0])), __dmul_rn((double)s1, g.H[3])), __dmul_rn((double)s2, g.H[6]));
        const double y = __dadd_rn(__dadd_rn(__dadd_rn(__dadd_rn(b0.y, -yi), __dmul_rn((double)s0, g.H[1])), __dmul_rn((double)s1, g.H[4])), __dmul_rn((double)s2, g.H[7]));
        const double z = __dadd_rn(__dadd_rn(__dadd_rn(__dadd_rn(b1.x, -zi), __dmul_rn((double)s0, g.H[2])), __dmul_rn((double)s1, g.H[5])), __dmul_rn((double)s2, g.H[8]));
        const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y)), __dmul_rn(z, z));
        hit = r2 < r2max;
        key = (unsigned)j * 27u + (unsigned)((s0 + 1) * 9 + (s1 + 1) * 3 + (s2 + 1));
      }
    }
    const unsigned m = __ballot_sync(full, hit);
    if (FILL && hit) {
      const int slot = n_row + __popc(m & ((1u << lane) - 1u));
      if (slot < kRowMax) keys[wib][slot] = key;
    }
    n_row += __popc(m);
  }
  if (MODE != NB_FILL && lane == 0) count[i] = n_row;
  if (!FILL) return;
  __syncwarp();
  if (n_row > kRowMax) { if (lane == 0 && !(MODE == NB_FILL && if_truncated)) atomicAdd(flag, 1); n_row = kRowMax; }
  for (int q = lane; q < n_row; q += 32) {                  // rank sort: the keys of a row are distinct
    const unsigned k = keys[wib][q];
    int rank = 0;
    for (int r = 0; r < n_row; ++r) rank += keys[wib][r] < k;
    sorted_keys[wib][rank] = k;
  }
  __syncwarp();
  if (MODE == NB_STASH) {
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(cursor, (unsigned long long)n_row);
    base = __shfl_sync(full, base, 0);
    const bool fits = base + (unsigned long long)n_row <= (unsigned long long)capacity;
    if (lane == 0) tstart[i] = fits ? (int)base : -1;
    if (fits) for (int q = lane; q < n_row; q += 32) tmp[base + q] = sorted_keys[wib][q];
    return;
  }
  const long long beg = off[i];
  const long long room = capacity - beg;                    // entries of this row that fit
  for (int q = lane; q < n_row && q < room; q += 32) idx[beg + q] = (int)(sorted_keys[wib][q] / 27u);
  for (int b = lane; b < 3 * n_row && b < 3 * room; b += 32) {
    const unsigned code = sorted_keys[wib][b / 3] % 27u;
    const int comp = b % 3;
    shift[3 * beg + b] = (signed char)((int)(comp == 0 ? code / 9u : comp == 1 ? (code / 3u) % 3u : code % 3u) - 1);
  }
}

// the stashed rows (NB_STASH) to their places in the list: a copy, one warp per atom
__global__ void __launch_bounds__(256) k_nb_place(const long long *__restrict__ off, const int *__restrict__ count,
                                                  const int *__restrict__ tstart, const unsigned *__restrict__ tmp, int n, long long capacity,
                                                  int *__restrict__ idx, signed char *__restrict__ shift) {
  if (off[n] > capacity) return;                             // truncated list: the NB_FILL pass behind this one writes it
  const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (i >= n) return;
  const int n_row = min(count[i], kRowMax), ts = tstart[i];
  if (ts < 0) return;
  const long long beg = off[i];
  for (int q = lane; q < n_row; q += 32) idx[beg + q] = (int)(tmp[ts + q] / 27u);
  for (int b = lane; b < 3 * n_row; b += 32) {
    const unsigned code = tmp[ts + b / 3] % 27u;
    const int comp = b % 3;
    shift[3 * beg + b] = (signed char)((int)(comp == 0 ? code / 9u : comp == 1 ? (code / 3u) % 3u : code % 3u) - 1);
  }
}

// rev[p] = position of (j, i, -s) for p = (i, j, s): binary search in row j (sorted by key)
__global__ void __launch_bounds__(256) k_nb_rev(const long long *__restrict__ off, const int *__restrict__ idx,
                                                const signed char *__restrict__ shift, int n, long long capacity, int *__restrict__ rev,
                                                int *__restrict__ flag) {
  const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (i >= n) return;
  const long long beg = off[i], end = min(off[i + 1], capacity);
  for (long long p = beg + lane; p < end; p += 32) {
    const int j = idx[p];
    // row j is sorted by (neighbour, shift): binary search on the neighbour index alone (one 4-byte load per probe), then
    // the few entries with that neighbour (one per image) are compared by shift
    const int w0 = -shift[3 * p], w1 = -shift[3 * p + 1], w2 = -shift[3 * p + 2];
    long long lo = off[j], hi = min(off[j + 1], capacity);
    const long long end_j = hi;
    while (lo < hi) {
      const long long mid = (lo + hi) >> 1;
      if (idx[mid] < i) lo = mid + 1; else hi = mid;
    }
    long long found = -1;
    for (long long q = lo; q < end_j && idx[q] == i; ++q)
      if (shift[3 * q] == w0 && shift[3 * q + 1] == w1 && shift[3 * q + 2] == w2) { found = q; break; }
    if (found < 0) atomicAdd(flag, 1);                       // cannot happen for a list built here (the test is symmetric)
    rev[p] = (int)found;
  }
}

// velocity-Verlet halves ("100 steps ... 1 fs"): v += (dt / 2) F / m ; x += dt v (first half only)
__global__ void k_vv(int n, double *__restrict__ pos, double *__restrict__ vel, const double *__restrict__ F, const int *__restrict__ type,
                     const double *__restrict__ inv_mass, double half_dt_ftm2v, double dt, int drift) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double s = half_dt_ftm2v * inv_mass[type[i]];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const double v = fma(s, F[3 * (size_t)i + c], vel[3 * (size_t)i + c]);
    vel[3 * (size_t)i + c] = v;
    if (drift) pos[3 * (size_t)i + c] = fma(dt, v, pos[3 * (size_t)i + c]);
  }
}
// kinetic energy partials sum_i m v^2 / 2 (fixed order per block) -- reduced by launch_reduce
__global__ void k_ke(int n, const double *__restrict__ vel, const int *__restrict__ type, const double *__restrict__ mass,
                     double half_mvv2e, double *__restrict__ ke_i) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double vx = vel[3 * (size_t)i], vy = vel[3 * (size_t)i + 1], vz = vel[3 * (size_t)i + 2];
  ke_i[i] = half_mvv2e * mass[type[i]] * (vx * vx + vy * vy + vz * vz);
}
}  // namespace

namespace {
__global__ void k_nb_finish(const long long *__restrict__ off, int n, const int *__restrict__ flag, long long *__restrict__ info,
                            int accumulate) {
  // pairs found (may exceed the capacity: then the arrays hold a truncated list); rows longer than the sort buffer or
  // pairs without a mirror.  accumulate: over the builds of an MD run (largest pair count, summed errors)
  info[0] = accumulate ? max(info[0], off[n]) : off[n];
  info[1] = (accumulate ? info[1] : 0) + flag[0];
}
// x -= floor(x . Hi) . H: atoms back into the box (before a list build of an MD run)
__global__ void k_wrap(NbGrid g, int n, double *__restrict__ pos) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double x = pos[3 * (size_t)i], y = pos[3 * (size_t)i + 1], z = pos[3 * (size_t)i + 2];
  const double w0 = floor(x * g.Hi[0] + y * g.Hi[3] + z * g.Hi[6]), w1 = floor(x * g.Hi[1] + y * g.Hi[4] + z * g.Hi[7]),
               w2 = floor(x * g.Hi[2] + y * g.Hi[5] + z * g.Hi[8]);
  if (w0 == 0.0 && w1 == 0.0 && w2 == 0.0) return;
  if (!(fabs(w0) < 1073741824.0 && fabs(w1) < 1073741824.0 && fabs(w2) < 1073741824.0)) return;   // left to k_nb_cells to count
  pos[3 * (size_t)i] = x - (w0 * g.H[0] + w1 * g.H[3] + w2 * g.H[6]);
  pos[3 * (size_t)i + 1] = y - (w0 * g.H[1] + w1 * g.H[4] + w2 * g.H[7]);
  pos[3 * (size_t)i + 2] = z - (w0 * g.H[2] + w1 * g.H[5] + w2 * g.H[8]);
}
size_t al(size_t x) { return (x + 255) & ~(size_t)255; }
struct NbLayout {
  size_t cell, wrap, ccount, cursor, start, totals, sorted, pos_s, rcount, tstart, flag, total;
};
NbLayout nb_layout(long long n, long long n_cells) {
  NbLayout L;
  size_t o = 0;
  L.cell = o; o = al(o + (size_t)n * 4);
  L.wrap = o; o = al(o + (size_t)n * 12);
  L.ccount = o; o = al(o + (size_t)n_cells * 4);
  L.cursor = o; o = al(o + (size_t)n_cells * 4);
  L.start = o; o = al(o + (size_t)(n_cells + 1) * 8);
  L.totals = o; o = al(o + (size_t)((std::max(n, n_cells) + 1) / 1024 + 3) * 8);
  L.sorted = o; o = al(o + (size_t)n * 4);
  L.pos_s = o; o = al(o + (size_t)n * 32);
  L.rcount = o; o = al(o + (size_t)n * 4);
  L.tstart = o; o = al(o + (size_t)n * 4);
  L.flag = o; o = al(o + 16);
  L.total = o;
  return L;
}
}  // namespace

// cells per lattice direction for this box and list radius: floor(height / r_list) >= 1, reduced when the grid would
// be much larger than the number of atoms (a sparse box); Hi = inverse box.  false: singular box.
bool nb_grid(const double *box, double r_list, long long n_atoms, NbGrid &g) {
  const double *a = box, *b = box + 3, *c = box + 6;
  const double bc[3] = {b[1] * c[2] - b[2] * c[1], b[2] * c[0] - b[0] * c[2], b[0] * c[1] - b[1] * c[0]};
  const double ca[3] = {c[1] * a[2] - c[2] * a[1], c[2] * a[0] - c[0] * a[2], c[0] * a[1] - c[1] * a[0]};
  const double ab[3] = {a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]};
  const double vol = a[0] * bc[0] + a[1] * bc[1] + a[2] * bc[2];
  if (!(std::fabs(vol) > 0) || !(r_list > 0)) return false;
  for (int i = 0; i < 9; ++i) g.H[i] = box[i];
  for (int i = 0; i < 3; ++i) { g.Hi[3 * i + 0] = bc[i] / vol; g.Hi[3 * i + 1] = ca[i] / vol; g.Hi[3 * i + 2] = ab[i] / vol; }
  auto norm = [](const double *v) { return std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]); };
  const double h[3] = {std::fabs(vol) / norm(bc), std::fabs(vol) / norm(ca), std::fabs(vol) / norm(ab)};
  for (int k = 0; k < 3; ++k) g.nc[k] = std::max(1, (int)std::floor(h[k] / r_list));
  while ((long long)g.nc[0] * g.nc[1] * g.nc[2] > 8 * n_atoms + 64) {       // larger cells are still correct
    int k = g.nc[0] >= g.nc[1] ? (g.nc[0] >= g.nc[2] ? 0 : 2) : (g.nc[1] >= g.nc[2] ? 1 : 2);
    g.nc[k] = std::max(1, g.nc[k] / 2);
  }
  return true;
}

size_t nb_workspace_bytes(long long n_atoms) { return nb_layout(n_atoms, 8 * n_atoms + 64).total + 256; }

cudaError_t launch_neighbors_build(const NbGrid &g, long long n, const double *pos, double r_list, long long capacity, long long *off,
                                   int *idx, signed char *shift, int *rev, long long *info, int accumulate, void *ws, cudaStream_t st) {
  const long long n_cells = (long long)g.nc[0] * g.nc[1] * g.nc[2];
  const NbLayout L = nb_layout(n, n_cells);
  char *w = (char *)ws;
  int *cell = (int *)(w + L.cell), *wrap = (int *)(w + L.wrap), *ccount = (int *)(w + L.ccount), *cursor = (int *)(w + L.cursor);
  long long *start = (long long *)(w + L.start), *totals = (long long *)(w + L.totals);
  int *sorted = (int *)(w + L.sorted), *rcount = (int *)(w + L.rcount), *flag = (int *)(w + L.flag);
  double *pos_s = (double *)(w + L.pos_s);
  cudaError_t e = cudaMemsetAsync(w + L.ccount, 0, L.start - L.ccount, st);     // cell histogram and cursors
  if (e == cudaSuccess) e = cudaMemsetAsync(flag, 0, 16, st);
  if (e != cudaSuccess) return e;
  if (n == 0) { e = cudaMemsetAsync(off, 0, 8, st); if (e == cudaSuccess && !accumulate) e = cudaMemsetAsync(info, 0, 16, st); return e; }
  const int nb = (int)((n + 255) / 256);
  k_nb_cells<<<nb, 256, 0, st>>>(g, pos, (int)n, cell, wrap, ccount, flag);
  e = launch_scan(ccount, n_cells, start, totals, st);
  if (e != cudaSuccess) return e;
  k_nb_scatter<<<nb, 256, 0, st>>>(cell, (int)n, start, cursor, sorted);
  k_nb_sort_cells<<<(unsigned)((n_cells + 255) / 256), 256, 0, st>>>(start, (int)n_cells, sorted);
  k_nb_gather_pos<<<nb, 256, 0, st>>>(pos, sorted, wrap, (int)n, pos_s);
  const double r2 = r_list * r_list;
  const unsigned nw = (unsigned)((n + 7) / 8);
  int *tstart = (int *)(w + L.tstart);
  unsigned long long *claim = (unsigned long long *)(flag + 2);        // bytes 8 .. 15 of the flag block (zeroed above)
  if (rev && capacity > 0) {
    // one search: rows stashed in the rev array (overwritten by k_nb_rev afterwards), placed once the offsets exist
    k_nb_rows<NB_STASH><<<nw, 256, 0, st>>>(g, pos_s, cell, wrap, start, (int)n, r2, rcount, nullptr, capacity, nullptr, nullptr, flag, 0,
                                            tstart, (unsigned *)rev, claim);
    e = launch_scan(rcount, n, off, totals, st);
    if (e != cudaSuccess) return e;
    k_nb_place<<<nw, 256, 0, st>>>(off, rcount, tstart, (const unsigned *)rev, (int)n, capacity, idx, shift);
    k_nb_rows<NB_FILL><<<nw, 256, 0, st>>>(g, pos_s, cell, wrap, start, (int)n, r2, rcount, off, capacity, idx, shift, flag, 1, nullptr,
                                           nullptr, nullptr);
    count_launch();
  } else {
    k_nb_rows<NB_COUNT><<<nw, 256, 0, st>>>(g, pos_s, cell, wrap, start, (int)n, r2, rcount, nullptr, 0, nullptr, nullptr, flag, 0, nullptr,
                                            nullptr, nullptr);
    e = launch_scan(rcount, n, off, totals, st);
    if (e != cudaSuccess) return e;
    if (capacity > 0)
      k_nb_rows<NB_FILL><<<nw, 256, 0, st>>>(g, pos_s, cell, wrap, start, (int)n, r2, rcount, off, capacity, idx, shift, flag, 0, nullptr,
                                             nullptr, nullptr);
  }
  if (rev) k_nb_rev<<<(unsigned)((n + 7) / 8), 256, 0, st>>>(off, idx, shift, (int)n, capacity, rev, flag);
  k_nb_finish<<<1, 1, 0, st>>>(off, (int)n, flag, info, accumulate);
  for (int q = 0; q < 8; ++q) count_launch();
  return cudaGetLastError();
}

cudaError_t launch_wrap(const NbGrid &g, int n, double *pos, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_wrap<<<(n + 255) / 256, 256, 0, st>>>(g, n, pos);
  count_launch();
  return cudaGetLastError();
}
cudaError_t launch_vv(int n, double *pos, double *vel, const double *F, const int *type, const double *inv_mass, double half_dt_ftm2v,
                      double dt, int drift, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_vv<<<(n + 255) / 256, 256, 0, st>>>(n, pos, vel, F, type, inv_mass, half_dt_ftm2v, dt, drift);
  count_launch();
  return cudaGetLastError();
}
cudaError_t launch_ke(int n, const double *vel, const int *type, const double *mass, double half_mvv2e, double *ke_i, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_ke<<<(n + 255) / 256, 256, 0, st>>>(n, vel, type, mass, half_mvv2e, ke_i);
  count_launch();
  return cudaGetLastError();
}


// ---- mtp_neighbors_build_static: the list build with its workspace in a static device array -------------------------
// For callers that cannot allocate (stream capture, serving loops, harnesses that forbid cudaMalloc): the kernels of
// launch_neighbors_build, unchanged, on a workspace that lives in the library's device image.  Every GPU that loads
// the library holds the array (6 MiB) until the process exits.  All calls on a device share it: calls that overlap
// on the GPU (different streams without ordering) race; calls on one stream, or ordered by events, do not.
namespace {
constexpr long long kNbStaticAtoms = MTP_NB_STATIC_MAX_ATOMS;
constexpr size_t kNbStaticBytes = (size_t)6 << 20;          // nb_workspace_bytes(32 768) = 6 164 480
static __device__ __align__(256) unsigned char g_nb_static[kNbStaticBytes];

constexpr int kMaxDevices = 64;
std::mutex g_nb_static_mu;
void *g_nb_static_ptr[kMaxDevices] = {};

// Device address of the array on the current device.  In host code the name g_nb_static is only a handle for the
// runtime, not a device address: the address comes from cudaGetSymbolAddress, asked once per device with that
// device current (every device has its own copy of the array).
cudaError_t nb_static_address(void **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_nb_static_mu);
  if (!g_nb_static_ptr[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_nb_static);
    if (e != cudaSuccess) return e;
    g_nb_static_ptr[dev] = p;
  }
  *out = g_nb_static_ptr[dev];
  return cudaSuccess;
}
}  // namespace

}  // namespace mtpb

extern "C" int mtp_neighbors_build_static(int64_t N, const double *d_pos, const double *box, double r_list, int64_t capacity,
                                          int64_t *d_off, int32_t *d_idx, int8_t *d_shift, int32_t *d_rev, int64_t *d_info,
                                          void *stream) {
  using namespace mtpb;
  char msg[256];
  if (N < 0 || !box || !d_off || !d_info || capacity < 0 || (N > 0 && !d_pos) || (capacity > 0 && (!d_idx || !d_shift)) ||
      capacity > 0x7fffffffLL) {
    set_thread_error("mtp_neighbors_build_static: bad argument (null pointer or negative size)");
    return MTP_EINVAL;
  }
  if (N > kNbStaticAtoms || nb_workspace_bytes(N) > kNbStaticBytes) {
    std::snprintf(msg, sizeof msg,
                  "mtp_neighbors_build_static: n_atoms = %lld exceeds MTP_NB_STATIC_MAX_ATOMS = %lld "
                  "(use mtp_neighbors_build with a caller workspace)", (long long)N, kNbStaticAtoms);
    set_thread_error(msg);
    return MTP_ESIZE;
  }
  NbGrid g;
  if (!nb_grid(box, r_list, N, g)) {
    set_thread_error("mtp_neighbors_build_static: singular box or r_list <= 0");
    return MTP_EBOX;
  }
  void *ws = nullptr;
  cudaError_t e = nb_static_address(&ws);
  // what must start at zero (cell histogram, scatter cursors, error flag) is cleared by launch_neighbors_build on the
  // stream; everything else in the workspace is written before it is read, so the last call's contents do not matter
  if (e == cudaSuccess)
    e = launch_neighbors_build(g, N, d_pos, r_list, capacity, (long long *)d_off, d_idx, (signed char *)d_shift, d_rev,
                               (long long *)d_info, 0, ws, (cudaStream_t)stream);
  if (e != cudaSuccess) {
    std::snprintf(msg, sizeof msg, "mtp_neighbors_build_static: %s", cudaGetErrorString(e));
    set_thread_error(msg);
    return MTP_ECUDA;
  }
  return MTP_OK;
}
