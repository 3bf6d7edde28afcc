// Small memory-bound kernels around the hot path: input packing (a1), deterministic force
// gather over the reverse-neighbour index (a8), fixed-order reductions of E, virial and B.
#include <cuda_runtime.h>

#include <cstdint>

#include <algorithm>
#include <atomic>

#include "kernels.h"
#include "pair_kernels.cuh"

namespace mtpb {

static std::atomic<long long> g_launches{0};
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }
long long launch_count() { return g_launches.load(std::memory_order_relaxed); }

// pos4[i] = (x, y, z, species): one aligned 32-byte sector per neighbour gather
__global__ void k_pack(const double *__restrict__ pos, const int *__restrict__ type, int n,
                       double *__restrict__ pos4) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double2 *o = reinterpret_cast<double2 *>(pos4) + 2 * (size_t)i;
  o[0] = make_double2(pos[3 * (size_t)i], pos[3 * (size_t)i + 1]);
  o[1] = make_double2(pos[3 * (size_t)i + 2], (double)type[i]);
}

// Packed neighbour word j | code << 27 (pair_kernels.cuh): one 4-byte load per pair in K1 / K3 instead of an index and
// three shift bytes, and the shift vector becomes a table lookup.  The word has room for shifts in {-1,0,1}^3 and
// indices below 2^27 only: anything else (and j outside [0, n_atoms)) is counted in flag[0] (MTP_INFO_INPUT_ERRORS) and
// the pair is dropped (word -1) instead of aliasing to another image or atom.
// k_pack_pairs_chunk does this for the pairs of one chunk of atoms [c0, c1): out[p - off[c0]] for p in [off[c0], off[c1]), at most cap
// of them (the excess is counted in flag[1]).  The pair range is read on the device: no host synchronisation.
// Bit (j >> tshift) of the touch bitmap (kTouchWords x 32 bits, tshift chosen so that all atoms fit) is set for every
// neighbour j of the chunk: the force assembly walks only blocks of rows that hold a neighbour in the chunk.
__global__ void __launch_bounds__(256) k_pack_pairs_chunk(const long long *__restrict__ off, int c0, int c1, const int *__restrict__ idx,
                                                          const signed char *__restrict__ shift, long long n_atoms, long long cap,
                                                          int *__restrict__ out, int *__restrict__ flag, unsigned *__restrict__ touch,
                                                          int tshift, int vec) {
  __shared__ unsigned bits[kTouchWords];             // this block's share of the touch bitmap: merged into the global one at the end
  for (int i = threadIdx.x; i < kTouchWords; i += blockDim.x) bits[i] = 0u;
  __syncthreads();
  const long long p0 = off[c0], n = off[c1] - p0;
  // four CONSECUTIVE pairs per thread, at absolute positions 4 g .. 4 g + 3: the indices come as one 16-byte load and
  // the twelve shift bytes as three 4-byte loads (the arrays are 16-byte aligned: checked by the launcher, which
  // otherwise asks for the scalar loads)
  const long long g0 = p0 >> 2, g1 = (p0 + n + 3) >> 2;
  for (long long g = g0 + (long long)blockIdx.x * blockDim.x + threadIdx.x; g < g1; g += (long long)gridDim.x * blockDim.x) {
    int j[4];
    unsigned sw[3] = {0u, 0u, 0u};
    const long long a = 4 * g;
    if (vec && a >= p0 && a + 4 <= p0 + n) {
      const int4 v = *reinterpret_cast<const int4 *>(idx + a);
      j[0] = v.x; j[1] = v.y; j[2] = v.z; j[3] = v.w;
      if (shift) {
        const unsigned *sp = reinterpret_cast<const unsigned *>(shift + 3 * a);
        sw[0] = sp[0]; sw[1] = sp[1]; sw[2] = sp[2];
      }
    } else {
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const long long p = a + u;
        j[u] = -1;
        if (p >= p0 && p < p0 + n) {
          j[u] = idx[p];
          if (shift) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
              const int byte = 3 * u + c;
              sw[byte >> 2] |= (unsigned)(unsigned char)shift[3 * p + c] << (8 * (byte & 3));
            }
          }
        }
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const long long q = a + u - p0;
      if (q < 0 || q >= n) continue;
      int sv[3];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const int byte = 3 * u + c;
        sv[c] = (int)(signed char)((sw[byte >> 2] >> (8 * (byte & 3))) & 0xffu);
      }
      const bool ok = j[u] >= 0 && j[u] < n_atoms && sv[0] >= -1 && sv[0] <= 1 && sv[1] >= -1 && sv[1] <= 1 && sv[2] >= -1 && sv[2] <= 1;
      int word = -1;
      if (!ok) atomicAdd(flag, 1);
      else {
        word = shift ? (int)((unsigned)j[u] | ((unsigned)shift_code(sv[0], sv[1], sv[2]) << kIdxBits)) : j[u];
        const int b = j[u] >> tshift;
        atomicOr(&bits[b >> 5], 1u << (b & 31));
      }
      if (out) {
        if (q < cap) out[q] = word;
        else atomicAdd(flag + 1, 1);
      }
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < kTouchWords; i += blockDim.x) if (bits[i]) atomicOr(touch + i, bits[i]);
}

// Live rows (MTP_OPT_SKIN_LIST; reading G3: listed pairs with r >= R_cut contribute exactly nothing): the packer of a
// list that carries a skin.  One warp per atom of the chunk: the row's entries within R_cut are moved to the front of
// the row's stretch of the word array (order kept), cnt[atom - c0] says how many, korig[] keeps each one's position
// in the CSR row (K3 writes the d4 record there, so the reverse gather is unchanged), and the d4 records of the
// dropped entries are zeroed here.  The distance is pair_vector's, the test K1 / K3 make themselves: an entry dropped
// here is one they would have multiplied by zero.  K1 / K3 then loop over cnt instead of the CSR row length -- with a
// 1 A skin at R_cut = 5 A that is 1 / 1.73 of the pairs.
__global__ void __launch_bounds__(256) k_pack_rows_live(const PairArgs a, const int *__restrict__ idx, const signed char *__restrict__ shift,
                                                        long long n_atoms, long long cap, int *__restrict__ out,
                                                        unsigned short *__restrict__ korig, int *__restrict__ cnt, double *__restrict__ d4,
                                                        unsigned *__restrict__ touch, int tshift) {
  __shared__ unsigned bits[kTouchWords];
  __shared__ __align__(16) double slut[kShiftLut];
  for (int i = threadIdx.x; i < kTouchWords; i += blockDim.x) bits[i] = 0u;
  if (threadIdx.x < 27) {
    const int q = (threadIdx.x + 13) % 27;                  // code -> position in the {-1,0,1}^3 list (as stage_coef)
    const double s0 = q / 9 - 1, s1 = (q / 3) % 3 - 1, s2 = q % 3 - 1;
    slut[4 * threadIdx.x] = s0 * a.H[0] + s1 * a.H[3] + s2 * a.H[6];
    slut[4 * threadIdx.x + 1] = s0 * a.H[1] + s1 * a.H[4] + s2 * a.H[7];
    slut[4 * threadIdx.x + 2] = s0 * a.H[2] + s1 * a.H[5] + s2 * a.H[8];
    slut[4 * threadIdx.x + 3] = 0.0;
  }
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const long long p0 = a.off[a.c0];
  const double rc2 = a.r_cut * a.r_cut;
  for (int i = a.c0 + ((blockIdx.x * blockDim.x + threadIdx.x) >> 5); i < a.c1; i += (gridDim.x * blockDim.x) >> 5) {
    const long long beg = a.off[i], rb = beg - p0;
    const int n = (int)min(a.off[i + 1] - beg, 65535LL);     // korig is 16 bits wide; longer rows are counted as errors below
    if (lane == 0 && a.off[i + 1] - beg > 65535LL) atomicAdd(a.flag, 1);
    double xi, yi, zi, ti;
    load_pos4(a.pos4, i, xi, yi, zi, ti);
    int live = 0;
    for (int base = 0; base < n; base += 32) {
      const int k = base + lane;
      bool keep = false;
      int word = -1, j = 0;
      const bool here = k < n && rb + k < cap;
      if (k < n && rb + k >= cap) atomicAdd(a.flag + 1, 1);
      if (here) {
        j = idx[beg + k];
        int s0 = 0, s1 = 0, s2 = 0;
        if (shift) { s0 = shift[3 * (beg + k)]; s1 = shift[3 * (beg + k) + 1]; s2 = shift[3 * (beg + k) + 2]; }
        const bool ok = j >= 0 && j < n_atoms && s0 >= -1 && s0 <= 1 && s1 >= -1 && s1 <= 1 && s2 >= -1 && s2 <= 1;
        if (!ok) atomicAdd(a.flag, 1);
        else {
          const int code = shift ? shift_code(s0, s1, s2) : 0;
          double xj, yj, zj, tj, x, y, z;
          load_pos4(a.pos4, j, xj, yj, zj, tj);
          pair_vector(a, slut, code, xi, yi, zi, xj, yj, zj, x, y, z);
          keep = x * x + y * y + z * z < rc2;
          word = (int)((unsigned)j | ((unsigned)code << kIdxBits));
        }
      }
      const unsigned m = __ballot_sync(0xffffffffu, keep);
      if (keep) {
        const int pos = live + __popc(m & ((1u << lane) - 1u));
        out[rb + pos] = word;
        korig[rb + pos] = (unsigned short)k;
        const int b = j >> tshift;
        atomicOr(&bits[b >> 5], 1u << (b & 31));
      } else if (here && d4) {
        double2 *o = reinterpret_cast<double2 *>(d4) + 2 * (size_t)(rb + k);
        o[0] = make_double2(0.0, 0.0); o[1] = make_double2(0.0, 0.0);
      }
      live += __popc(m);
    }
    if (lane == 0) cnt[i - a.c0] = live;
  }
  __syncthreads();
  for (int i = threadIdx.x; i < kTouchWords; i += blockDim.x) if (bits[i]) atomicOr(touch + i, bits[i]);
}

// G of a partitioned table before the group programs accumulate into it: dE_i/d(cut) for the packed moments
// that are cut nodes themselves (gmap[k] = their cut row), 0 for the others
__global__ void k_ginit(double *__restrict__ G, int n_cut_rows, int n_basic, int ncol, const int *__restrict__ gmap,
                        const double *__restrict__ Sbar) {
  const int col = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y;
  if (col >= ncol || k >= n_basic) return;
  const int r = gmap[k];
  G[tiled_index(n_basic, k, col)] = r >= 0 ? Sbar[tiled_index(n_cut_rows, r, col)] : 0.0;
}

// cut values of the packed moments that are cut nodes themselves: S[gmap[k]][:] = M[k][:]
__global__ void k_scopy(double *__restrict__ S, int n_cut_rows, int n_basic, int ncol, const int *__restrict__ gmap,
                        const double *__restrict__ M) {
  const int col = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y;
  if (col >= ncol || k >= n_basic) return;
  const int r = gmap[k];
  if (r >= 0) S[tiled_index(n_cut_rows, r, col)] = M[tiled_index(n_basic, k, col)];
}

// tiled [tiles][rows][128] -> row-major dst[row * ld + col], or its transpose dst[col * ld + row]
__global__ void k_untile(const double *__restrict__ src, int rows, long long ncol, double *__restrict__ dst, long long ld,
                         int transpose) {
  const long long col = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int row = blockIdx.y;
  if (col >= ncol || row >= rows) return;
  const double v = src[tiled_index(rows, row, col)];
  if (transpose) dst[col * ld + row] = v; else dst[(long long)row * ld + col] = v;
}

// Prologue of mtp_compute in one launch (small systems pay per launch): pos4 = (x, y, z, species), F = 0, the virial
// partials = 0, the touch bitmap of the first chunk = 0
__global__ void k_prologue(const double *__restrict__ pos, const int *__restrict__ type, int n, double *__restrict__ pos4,
                           double *__restrict__ F, double *__restrict__ wpart, long long n_wpart, unsigned *__restrict__ touch) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) {
    double2 *o = reinterpret_cast<double2 *>(pos4) + 2 * (size_t)i;
    o[0] = make_double2(pos[3 * (size_t)i], pos[3 * (size_t)i + 1]);
    o[1] = make_double2(pos[3 * (size_t)i + 2], (double)type[i]);
    F[3 * (size_t)i] = 0.0; F[3 * (size_t)i + 1] = 0.0; F[3 * (size_t)i + 2] = 0.0;
  }
  if (i < n_wpart) wpart[i] = 0.0;
  if (i < kTouchWords) touch[i] = 0u;
}

__global__ void k_zero(double *p, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = 0.0;
}

// a8 with bounded per-pair scratch (SURVEY.md 8(a) note on a8 + a10, design (ii)): the pair kernel of the chunk
// [c0, c1) has written d4[p - off[c0]] for the chunk's pairs and added each atom's own sum to F; here every atom k
// with a neighbour j in the chunk subtracts d_jk, found through rev.  One warp per atom, lanes over the row,
// xor-shuffle tree, one read-modify-write of F_k per chunk: the chunks come in stream order, so the sum has a fixed
// order and is bit-reproducible (G19).  Blocks of 2^tshift rows without a neighbour in the chunk (touch bitmap
// written by k_pack_pairs_chunk) are skipped without reading their rows.
__global__ void __launch_bounds__(256) k_gather_chunk(const long long *__restrict__ off, const int *__restrict__ idx,
                                                      const int *__restrict__ rev, const double *__restrict__ d4, long long d4_cap,
                                                      int c0, int c1, int n_atoms, const unsigned *__restrict__ touch, int tshift,
                                                      double *__restrict__ F) {
  const int lane = threadIdx.x & 31;
  // the mirror pair of p lies in this chunk exactly when rev[p] falls into the chunk's pair range: idx is not read
  const long long p0 = off[c0], np = off[c1] - p0;
  const double2 *d = reinterpret_cast<const double2 *>(d4);
  for (int k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; k < n_atoms; k += (gridDim.x * blockDim.x) >> 5) {
    if (!((touch[(k >> tshift) >> 5] >> ((k >> tshift) & 31)) & 1u)) continue;
    const long long beg = off[k], end = off[k + 1];
    double fx = 0, fy = 0, fz = 0;
    bool any = false;
    for (long long p = beg + lane; p < end; p += 32) {
      const long long q = rev[p] - p0;
      if (q >= 0 && q < np) {
        if (q < d4_cap) {
          const double2 b0 = __ldg(d + 2 * q), b1 = __ldg(d + 2 * q + 1);
          fx -= b0.x; fy -= b0.y; fz -= b1.x;
        }
        any = true;
      }
    }
    any = __any_sync(0xffffffffu, any);
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
      fx += __shfl_xor_sync(0xffffffffu, fx, o);
      fy += __shfl_xor_sync(0xffffffffu, fy, o);
      fz += __shfl_xor_sync(0xffffffffu, fz, o);
    }
    if (lane == 0 && any) { F[3 * (size_t)k] += fx; F[3 * (size_t)k + 1] += fy; F[3 * (size_t)k + 2] += fz; }
  }
}

// out[blockIdx.x][c] = sum over this block's share of i of in[i*stride + c], c < ncomp <= 8.
// Fixed grid, fixed order -> bit-reproducible.  Two launches reduce any n: kReduceBlocks partial rows
// of stride 8, then one block over those.
constexpr int kReduceBlocks = 256;
__global__ void __launch_bounds__(1024) k_reduce_rows(const double *__restrict__ in, long long n, int stride,
                                                      int ncomp, double *__restrict__ out) {
  __shared__ double sm[32][8];
  double acc[8];
#pragma unroll
  for (int c = 0; c < 8; ++c) acc[c] = 0.0;
  for (long long i = (long long)blockIdx.x * 1024 + threadIdx.x; i < n; i += 1024LL * gridDim.x)
    for (int c = 0; c < ncomp; ++c) acc[c] += in[i * stride + c];
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    double v = acc[c];
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5][c] = v;
  }
  __syncthreads();
  if (threadIdx.x < 8) {
    double v = 0.0;
    if (threadIdx.x < ncomp)
      for (int w = 0; w < 32; ++w) v += sm[w][threadIdx.x];
    if (gridDim.x > 1) out[(size_t)blockIdx.x * 8 + threadIdx.x] = v;
    else if (threadIdx.x < ncomp) out[threadIdx.x] = v;
  }
}

// Bsum[b] += sum_i Bt[b][i] over the tiled Bt of a chunk: one warp per b, lanes stride the atoms, xor-shuffle tree
// (fixed order -> bit-reproducible); accumulates across chunks in launch order
__global__ void __launch_bounds__(256) k_colsum(const double *__restrict__ Bt, long long n, int nb, double *__restrict__ Bsum) {
  const int b = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (b >= nb) return;
  double acc = 0.0;
  for (long long i = lane; i < n; i += 32) acc += Bt[tiled_index(nb, b, i)];
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) Bsum[b] += acc;
}

cudaError_t launch_pack(const double *pos, const int *type, int n, double *pos4, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_pack<<<(n + 255) / 256, 256, 0, st>>>(pos, type, n, pos4);
  count_launch();
  return cudaGetLastError();
}
cudaError_t launch_untile(const double *src, int rows, long long ncol, double *dst, long long ld, int transpose, cudaStream_t st) {
  if (ncol <= 0 || rows <= 0) return cudaSuccess;
  k_untile<<<dim3((unsigned)((ncol + 127) / 128), rows), 128, 0, st>>>(src, rows, ncol, dst, ld, transpose);
  count_launch();
  return cudaGetLastError();
}
cudaError_t launch_ginit(double *G, int n_cut_rows, int n_basic, int ncol, const int *gmap, const double *Sbar,
                         cudaStream_t st) {
  if (ncol <= 0 || n_basic <= 0) return cudaSuccess;
  k_ginit<<<dim3((ncol + 255) / 256, n_basic), 256, 0, st>>>(G, n_cut_rows, n_basic, ncol, gmap, Sbar);
  count_launch();
  return cudaGetLastError();
}
cudaError_t launch_scopy(double *S, int n_cut_rows, int n_basic, int ncol, const int *gmap, const double *M, cudaStream_t st) {
  if (ncol <= 0 || n_basic <= 0) return cudaSuccess;
  k_scopy<<<dim3((ncol + 255) / 256, n_basic), 256, 0, st>>>(S, n_cut_rows, n_basic, ncol, gmap, M);
  count_launch();
  return cudaGetLastError();
}
cudaError_t launch_prologue(const double *pos, const int *type, int n, double *pos4, double *F, double *wpart, long long n_wpart,
                            unsigned *touch, cudaStream_t st) {
  const long long m = std::max<long long>(std::max<long long>(n, n_wpart), kTouchWords);
  k_prologue<<<(unsigned)((m + 255) / 256), 256, 0, st>>>(pos, type, n, pos4, F, wpart, n_wpart, touch);
  count_launch();
  return cudaGetLastError();
}
cudaError_t launch_zero(double *p, long long n, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_zero<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(p, n);
  count_launch();
  return cudaGetLastError();
}
cudaError_t launch_pack_pairs_chunk(const long long *off, int c0, int c1, const int *idx, const signed char *shift, long long n_atoms,
                                    long long cap, int *out, int *flag, unsigned *touch, cudaStream_t st, bool touch_is_zero) {
  if (c1 <= c0) return cudaSuccess;
  cudaError_t e = touch_is_zero ? cudaSuccess : cudaMemsetAsync(touch, 0, kTouchWords * sizeof(unsigned), st);
  if (e != cudaSuccess) return e;
  // the pair count of the chunk lives on the device: a persistent grid strides over it
  const long long blocks = std::min<long long>(148 * 8, std::max<long long>(1, (cap + 1023) / 1024));
  const int vec = (((uintptr_t)idx & 15) == 0 && ((uintptr_t)shift & 3) == 0) ? 1 : 0;
  k_pack_pairs_chunk<<<(unsigned)blocks, 256, 0, st>>>(off, c0, c1, idx, shift, n_atoms, cap, out, flag, touch, touch_shift(n_atoms), vec);
  count_launch();
  return cudaGetLastError();
}
cudaError_t launch_pack_rows_live(const PairArgs &a, const int *idx, const signed char *shift, long long n_atoms, long long cap, int *out,
                                  unsigned short *korig, int *cnt, double *d4, unsigned *touch, cudaStream_t st, bool touch_is_zero) {
  if (a.c1 <= a.c0) return cudaSuccess;
  cudaError_t e = touch_is_zero ? cudaSuccess : cudaMemsetAsync(touch, 0, kTouchWords * sizeof(unsigned), st);
  if (e != cudaSuccess) return e;
  const int blocks = (int)std::min<long long>(148 * 8, ((long long)(a.c1 - a.c0) + 7) / 8);
  k_pack_rows_live<<<blocks, 256, 0, st>>>(a, idx, shift, n_atoms, cap, out, korig, cnt, d4, touch, touch_shift(n_atoms));
  count_launch();
  return cudaGetLastError();
}
cudaError_t launch_gather_chunk(const long long *off, const int *idx, const int *rev, const double *d4, long long d4_cap, int c0,
                                int c1, int n_atoms, const unsigned *touch, double *F, cudaStream_t st) {
  if (c1 <= c0) return cudaSuccess;
  k_gather_chunk<<<148 * 8, 256, 0, st>>>(off, idx, rev, d4, d4_cap, c0, c1, n_atoms, touch, touch_shift(n_atoms), F);
  count_launch();
  return cudaGetLastError();
}
cudaError_t launch_reduce(const double *in, long long n, int stride, int ncomp, double *out, double *scratch,
                          cudaStream_t st) {
  if (n > 4 * 1024 && scratch) {          // one block alone is latency-bound: 82 us for the 32 768 virial partials of config 4
    k_reduce_rows<<<kReduceBlocks, 1024, 0, st>>>(in, n, stride, ncomp, scratch);
    count_launch();
    k_reduce_rows<<<1, 1024, 0, st>>>(scratch, kReduceBlocks, 8, ncomp, out);
  } else {
    k_reduce_rows<<<1, 1024, 0, st>>>(in, n, stride, ncomp, out);
  }
  count_launch();
  return cudaGetLastError();
}
// E = sum E_i and the six virial sums in the same launches: blockIdx.y selects the array (fixed order, as launch_reduce)
__global__ void __launch_bounds__(1024) k_reduce_two(const double *__restrict__ in0, long long n0, int stride0, int ncomp0, double *__restrict__ out0,
                                                     const double *__restrict__ in1, long long n1, int stride1, int ncomp1,
                                                     double *__restrict__ out1) {
  const bool second = blockIdx.y == 1;
  const double *in = second ? in1 : in0;
  const long long n = second ? n1 : n0;
  const int stride = second ? stride1 : stride0, ncomp = second ? ncomp1 : ncomp0;
  double *out = second ? out1 : out0;
  __shared__ double sm[32][8];
  double acc[8];
#pragma unroll
  for (int c = 0; c < 8; ++c) acc[c] = 0.0;
  for (long long i = (long long)blockIdx.x * 1024 + threadIdx.x; i < n; i += 1024LL * gridDim.x)
    for (int c = 0; c < ncomp; ++c) acc[c] += in[i * stride + c];
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    double v = acc[c];
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5][c] = v;
  }
  __syncthreads();
  if (threadIdx.x < 8) {
    double v = 0.0;
    if (threadIdx.x < ncomp)
      for (int w = 0; w < 32; ++w) v += sm[w][threadIdx.x];
    if (gridDim.x > 1) out[(size_t)blockIdx.x * 8 + threadIdx.x] = v;
    else if (threadIdx.x < ncomp) out[threadIdx.x] = v;
  }
}
// E (from Ei [n]) and, when virial != null, the virial (from wpart [n_w][8]); scratch: 2 x kReduceBlocks x 8 doubles.
// The same summation order as two launch_reduce calls.
cudaError_t launch_reduce_energy_virial(const double *Ei, long long n, double *E, const double *wpart, long long n_w, double *virial,
                                        double *scratch, cudaStream_t st) {
  const dim3 two(1, virial ? 2 : 1);
  if (std::max(n, virial ? n_w : 0) > 4 * 1024) {
    // level 1 writes kReduceBlocks partial rows per array (an array shorter than the grid just leaves zeros), level 2 sums them
    double *s0 = scratch, *s1 = scratch + kReduceBlocks * 8;
    k_reduce_two<<<dim3(kReduceBlocks, two.y), 1024, 0, st>>>(Ei, n, 1, 1, s0, wpart, n_w, 8, 6, s1);
    count_launch();
    k_reduce_two<<<two, 1024, 0, st>>>(s0, kReduceBlocks, 8, 1, E, s1, kReduceBlocks, 8, 6, virial);
  } else {
    k_reduce_two<<<two, 1024, 0, st>>>(Ei, n, 1, 1, E, wpart, n_w, 8, 6, virial);
  }
  count_launch();
  return cudaGetLastError();
}
cudaError_t launch_colsum(const double *Bt, long long n, int nb, double *Bsum, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_colsum<<<(nb + 7) / 8, 256, 0, st>>>(Bt, n, nb, Bsum);
  count_launch();
  return cudaGetLastError();
}

}  // namespace mtpb
