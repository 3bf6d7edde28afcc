// Small memory-bound kernels around the hot path: input packing (a1), deterministic force
// gather over the reverse-neighbour index (a8), fixed-order reductions of E, virial and B.
#include <cuda_runtime.h>

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

// packed neighbour word j | code << 27 (pair_kernels.cuh): one 4-byte load per pair in K1 / K3 instead of
// an index and three shift bytes, and the shift vector becomes a table lookup.  The word has room for shifts in
// {-1,0,1}^3 and indices below 2^27 only: anything else (and j outside [0, n_atoms)) is counted in *flag
// (MTP_INFO_INPUT_ERRORS) and the pair is dropped (word -1) instead of aliasing to another image or atom.
__global__ void k_pack_pairs(const int *__restrict__ idx, const signed char *__restrict__ shift, long long nnz,
                             long long n_atoms, int *__restrict__ out, int *__restrict__ flag) {
  const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= nnz) return;
  const int s0 = shift[3 * p], s1 = shift[3 * p + 1], s2 = shift[3 * p + 2], j = idx[p];
  const bool ok = s0 >= -1 && s0 <= 1 && s1 >= -1 && s1 <= 1 && s2 >= -1 && s2 <= 1 && j >= 0 && j < n_atoms;
  if (!ok) { atomicAdd(flag, 1); out[p] = -1; return; }
  out[p] = (int)((unsigned)j | ((unsigned)shift_code(s0, s1, s2) << kIdxBits));
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

__global__ void k_zero(double *p, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = 0.0;
}

// a8 gather: F_k = sum_{p in row k} ( d[p] - d[rev[p]] ); one warp per atom, lanes over the
// row, xor-shuffle tree -> the summation order is fixed, the result bit-reproducible (G19).
__global__ void __launch_bounds__(256) k_gather(const long long *__restrict__ off, const int *__restrict__ rev,
                                                const double *__restrict__ d4, int n, double *__restrict__ F) {
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= n) return;
  const long long beg = off[warp], end = off[warp + 1];
  double fx = 0, fy = 0, fz = 0;
  const double2 *d = reinterpret_cast<const double2 *>(d4);
  for (long long p = beg + lane; p < end; p += 32) {
    const long long q = rev[p];
    const double2 a0 = d[2 * p], a1 = d[2 * p + 1];
    const double2 b0 = __ldg(d + 2 * q), b1 = __ldg(d + 2 * q + 1);
    fx += a0.x - b0.x; fy += a0.y - b0.y; fz += a1.x - b1.x;
  }
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) {
    fx += __shfl_xor_sync(0xffffffffu, fx, o);
    fy += __shfl_xor_sync(0xffffffffu, fy, o);
    fz += __shfl_xor_sync(0xffffffffu, fz, o);
  }
  if (lane == 0) { F[3 * (size_t)warp] = fx; F[3 * (size_t)warp + 1] = fy; F[3 * (size_t)warp + 2] = fz; }
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
cudaError_t launch_pack_pairs(const int *idx, const signed char *shift, long long nnz, long long n_atoms, int *out, int *flag,
                              cudaStream_t st) {
  if (nnz <= 0) return cudaSuccess;
  k_pack_pairs<<<(unsigned)((nnz + 255) / 256), 256, 0, st>>>(idx, shift, nnz, n_atoms, out, flag);
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
cudaError_t launch_zero(double *p, long long n, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_zero<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(p, n);
  count_launch();
  return cudaGetLastError();
}
cudaError_t launch_gather(const long long *off, const int *rev, const double *d4, int n, double *F,
                          cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_gather<<<(n + 7) / 8, 256, 0, st>>>(off, rev, d4, n, F);
  count_launch();
  return cudaGetLastError();
}
cudaError_t launch_reduce(const double *in, long long n, int stride, int ncomp, double *out, double *scratch,
                          cudaStream_t st) {
  if (n > 64 * 1024 && scratch) {
    k_reduce_rows<<<kReduceBlocks, 1024, 0, st>>>(in, n, stride, ncomp, scratch);
    count_launch();
    k_reduce_rows<<<1, 1024, 0, st>>>(scratch, kReduceBlocks, 8, ncomp, out);
  } else {
    k_reduce_rows<<<1, 1024, 0, st>>>(in, n, stride, ncomp, out);
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
