// K5 (a9): extrapolation grades.  gamma_i = max_k | sum_a B[i][a] Ainv[a][k] |  (PAPER.md:35,46
// neighbourhood mode) and gamma = max_k | (sum_i B_i) Ainv |_k (configuration mode).
// BASELINE.json north_star: "a batched B.A^-1 grade kernel, the one genuinely dense
// contraction".  fp64 has no tcgen05 kind; this is a GEMM on the fp64 tensor-core path that does
// exist (mma.sync m8n8k4, 128x64x16 CTA tile) whose epilogue folds |.| and the row maximum, so the
// N x n_basis product is never written.  Non-negative doubles order like their bit patterns, so the row
// maximum across column tiles is an integer atomicMax (order independent -> deterministic).
#include <cuda_runtime.h>

#include <algorithm>

#include "kernels.h"

namespace mtpb {

constexpr int GBM = 128, GBN = 64, GBK = 16;
constexpr int GLDA = GBM + 8, GLDB = GBN + 4;   // strides = 8 / 4 mod 16 doubles: the mma fragment loads are conflict-free

// One fp64 tensor-core MMA (the only fp64 MMA on sm_100: legacy mma.sync, no tcgen05 kind): D(8x8) += A(8x4) B(4x8).
// Fragments: lane l holds A[l/4][l%4], B[l%4][l/4], C[l/4][2(l%4) + {0,1}].  Measured 37.1 TFLOP/s = the DFMA
// peak, at 1/8 of the instruction issues and with each shared-memory operand feeding 8 FMAs.
__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// CTA tile 128 atoms x 64 columns, 8 warps (4 x 2), warp tile 32 x 32 = 4 x 4 MMA tiles.
// B arrives as the tiled Bt [tile of 128 atoms][nb][128] the K2 kernels write (kTile = GBM): a CTA's A tile is one
// contiguous run of 128 atoms per k, kept k-major in shared memory.
__global__ void __launch_bounds__(256) k_grade(const double *__restrict__ Bt, const double *__restrict__ Ainv,
                                               long long n, int nb, double *__restrict__ gamma) {
  __shared__ __align__(16) double As[GBK][GLDA];     // B values of the tile, [k][atom]
  __shared__ __align__(16) double Bs[GBK][GLDB];     // Ainv rows of the tile, [k][column]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = (warp & 3) * 32, wn = (warp >> 2) * 32;
  const int fr = lane >> 2, fc = lane & 3;
  const long long m0 = (long long)blockIdx.y * GBM;
  const int n0 = blockIdx.x * GBN;
  double acc[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }
  const int arow = tid & 127, ak = (tid >> 7) * 8;      // A tile: 16 k x 128 atoms, consecutive threads = consecutive atoms
  const double *Btile = Bt + (size_t)blockIdx.y * nb * GBM;
  const int bk = tid >> 4, bc = (tid & 15) * 4;         // Ainv tile: 16 k x 64 cols
  for (int k0 = 0; k0 < nb; k0 += GBK) {
    {
      const long long row = m0 + arow;
#pragma unroll
      for (int j = 0; j < 8; ++j) As[ak + j][arow] = (row < n && k0 + ak + j < nb) ? Btile[(size_t)(k0 + ak + j) * GBM + arow] : 0.0;
      const int kr = k0 + bk;
      const double *s2 = Ainv + (long long)kr * nb + n0 + bc;
#pragma unroll
      for (int j = 0; j < 4; ++j) Bs[bk][bc + j] = (kr < nb && n0 + bc + j < nb) ? s2[j] : 0.0;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < GBK; kk += 4) {
      double a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = As[kk + fc][wm + 8 * i + fr];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Bs[kk + fc][wn + 8 * j + fr];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    double m = 0.0;
#pragma unroll
    for (int j = 0; j < 4; ++j) m = fmax(m, fmax(fabs(acc[i][j][0]), fabs(acc[i][j][1])));
    m = fmax(m, __shfl_xor_sync(0xffffffffu, m, 1));
    m = fmax(m, __shfl_xor_sync(0xffffffffu, m, 2));
    const long long row = m0 + wm + 8 * i + fr;
    if (fc == 0 && row < n)
      atomicMax(reinterpret_cast<unsigned long long *>(gamma) + row, (unsigned long long)__double_as_longlong(m));
  }
}

// configuration mode: y_k = sum_a Bsum[a] Ainv[a][k]; gamma = max_k |y_k|
__global__ void k_grade_cfg(const double *__restrict__ Bsum, const double *__restrict__ Ainv, int nb,
                            double *__restrict__ gamma_cfg) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  double y = 0.0;
  if (k < nb)
    for (int a = 0; a < nb; ++a) y = fma(Bsum[a], Ainv[(long long)a * nb + k], y);
  double m = fabs(y);
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0)
    atomicMax(reinterpret_cast<unsigned long long *>(gamma_cfg), (unsigned long long)__double_as_longlong(m));
}

cudaError_t launch_grade(const double *Bt, const double *Ainv, long long n, int nb, double *gamma, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  cudaError_t e = launch_zero(gamma, n, st);
  if (e != cudaSuccess) return e;
  dim3 g((nb + GBN - 1) / GBN, (unsigned)((n + GBM - 1) / GBM));
  static_assert(GBM == kTile, "the CTA tile is one tile of the Bt layout");
  k_grade<<<g, 256, 0, st>>>(Bt, Ainv, n, nb, gamma);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_grade_cfg(const double *Bsum, const double *Ainv, int nb, double *scratch, double *gamma_cfg,
                             cudaStream_t st) {
  (void)scratch;
  cudaError_t e = launch_zero(gamma_cfg, 1, st);
  if (e != cudaSuccess) return e;
  k_grade_cfg<<<(nb + 127) / 128, 128, 0, st>>>(Bsum, Ainv, nb, gamma_cfg);
  count_launch();
  return cudaGetLastError();
}

// maximum of n non-negative doubles (the neighbourhood grades of a configuration): integer atomicMax on the bit
// pattern, order independent -> deterministic
__global__ void k_max_nonneg(const double *__restrict__ x, long long n, double *__restrict__ out) {
  double m = 0.0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) m = fmax(m, x[i]);
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m > 0.0) atomicMax(reinterpret_cast<unsigned long long *>(out), (unsigned long long)__double_as_longlong(m));
}
cudaError_t launch_max_nonneg(const double *x, long long n, double *out, cudaStream_t st) {
  cudaError_t e = launch_zero(out, 1, st);
  if (e != cudaSuccess || n <= 0) return e;
  const int blocks = (int)std::min<long long>((n + 255) / 256, 148 * 8);
  k_max_nonneg<<<blocks, 256, 0, st>>>(x, n, out);
  count_launch();
  return cudaGetLastError();
}

// ---- fp64 FMA throughput: 8 independent chains per thread, 4 blocks of 256 threads per SM
__global__ void __launch_bounds__(256) k_peak_dfma(long long iters, double *sink) {
  double a0 = 1.0 + threadIdx.x * 1e-9, a1 = a0 + 1e-3, a2 = a0 + 2e-3, a3 = a0 + 3e-3;
  double a4 = a0 + 4e-3, a5 = a0 + 5e-3, a6 = a0 + 6e-3, a7 = a0 + 7e-3;
  const double m = 0.999999, c = 1e-7;
  for (long long i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
      a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
  }
  const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
  if (s == 123.456) sink[0] = s;
}

cudaError_t launch_peak_dfma(long long iters, double *sink, double *flops_out, cudaStream_t st) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int grid = sms * 4;
  k_peak_dfma<<<grid, 256, 0, st>>>(iters, sink);
  count_launch();
  if (flops_out) *flops_out = 2.0 * 64.0 * (double)iters * 256.0 * grid;
  return cudaGetLastError();
}

}  // namespace mtpb
