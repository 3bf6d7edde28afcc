// Device helpers shared by the pair kernels K1 / K3 (pair_tiled.cuh): a1 pair geometry, a2 + a3
// Chebyshev radial basis and species-pair radial functions, small powers.  BASELINE.json
// north_star; readings G1-G7, G17 in DESIGN.md.  All arithmetic is on the DFMA pipe.
#pragma once
#include <cuda_runtime.h>
#include "stair.h"
#include "pair_kernels_args.h"

namespace mtpb {


__device__ __forceinline__ void pow_small(int s, double y, double &p, double &dp) {
  p = 1.0; dp = 0.0;
  if (s == 1) { p = y; dp = 1.0; }
  else if (s == 2) { p = y * y; dp = 2.0 * y; }
  else if (s == 3) { double y2 = y * y; p = y2 * y; dp = 3.0 * y2; }
}
template <int N>
__device__ __forceinline__ void pow_fixed(double y, double &p, double &dp) {
  if (N == 1) { p = y; dp = 1.0; }
  else if (N == 2) { p = y * y; dp = 2.0 * y; }
  else { double y2 = y * y; p = y2 * y2; dp = 4.0 * y2 * y; }
}

// a2 + a3: f_mu(r) = (R_cut - r)^2 sum_b c[mu][b] T_b(xi),  xi = (2r - R_min - R_cut)/(R_cut - R_min).
// crow points at the (z_i, z_j) block of the staged coefficients, laid out [b][NMUP] (NMUP = NMU rounded
// up to even) so that the coefficients of one b are read as 16-byte pairs.  NB > 0: compile-time basis
// size (8 in every BASELINE config), NB = 0: run-time nb.
template <int NMU, bool DERIV, int NB>
__device__ __forceinline__ void radial(const double *__restrict__ crow, int nb_rt, double r, double r_min,
                                       double r_cut, double inv_width, double *f, double *df) {
  constexpr int NMUP = (NMU + 1) & ~1;
  const int nb = NB > 0 ? NB : nb_rt;
  const double sx = 2.0 * inv_width;                     // inv_width = 1 / (R_cut - R_min), from the host
  const double xi = (2.0 * r - r_min - r_cut) * inv_width;
  double s[NMUP], ds[NMUP];
#pragma unroll
  for (int m = 0; m < NMUP; ++m) { s[m] = 0.0; ds[m] = 0.0; }
  double tm = 1.0, t = xi, dtm = 0.0, dt = 1.0;   // T_{b}, T_{b+1} and derivatives wrt xi
  const double2 *c2 = reinterpret_cast<const double2 *>(crow);
#pragma unroll
  for (int b = 0; b < nb; ++b) {
#pragma unroll
    for (int m = 0; m < NMUP; m += 2) {
      const double2 c = c2[(b * NMUP + m) >> 1];
      // T_0 = 1, T_0' = 0, T_1' = 1 written out (same values, no multiplications by 0 and 1 on the fp64 pipe)
      if (b == 0) { s[m] = c.x; s[m + 1] = c.y; }
      else { s[m] = fma(c.x, tm, s[m]); s[m + 1] = fma(c.y, tm, s[m + 1]); }
      if (DERIV) {
        if (b == 1) { ds[m] = c.x; ds[m + 1] = c.y; }
        else if (b > 1) { ds[m] = fma(c.x, dtm, ds[m]); ds[m + 1] = fma(c.y, dtm, ds[m + 1]); }
      }
    }
    const double tn = fma(2.0 * xi, t, -tm);
    if (DERIV) { const double dtn = fma(2.0 * xi, dt, fma(2.0, t, -dtm)); dtm = dt; dt = dtn; }
    tm = t; t = tn;
  }
  const double cut = r_cut - r, s2 = cut * cut;
#pragma unroll
  for (int m = 0; m < NMU; ++m) {
    f[m] = s[m] * s2;
    if (DERIV) df[m] = fma(ds[m] * sx, s2, -2.0 * cut * s[m]);
  }
}

// Packed neighbour word (k_pack_pairs): bits 0..26 the neighbour index j, bits 27..31 the image code:
// 0 = no shift, c > 0 = shift number (c + 12) mod 27 of the list s = (q/9 - 1, (q/3)%3 - 1, q%3 - 1).
constexpr int kIdxBits = 27;
constexpr int kIdxMask = (1 << kIdxBits) - 1;
__host__ __device__ __forceinline__ int shift_code(int s0, int s1, int s2) {
  return ((s0 + 1) * 9 + (s1 + 1) * 3 + (s2 + 1) + 27 - 13) % 27;
}

// a1: r_ij = x_j - x_i + s.H (s.H from the 27-entry table in shared memory), then the minimum image
// when the caller gave no shifts
__device__ __forceinline__ void pair_vector(const PairArgs &a, const double *__restrict__ slut, int code, double xi,
                                            double yi, double zi, double xj, double yj, double zj, double &x, double &y,
                                            double &z) {
  const double2 s01 = *reinterpret_cast<const double2 *>(slut + 4 * code);
  x = (xj - xi) + s01.x; y = (yj - yi) + s01.y; z = (zj - zi) + slut[4 * code + 2];
  if (a.minimg) {
    const double f0 = rint(x * a.Hi[0] + y * a.Hi[3] + z * a.Hi[6]);
    const double f1 = rint(x * a.Hi[1] + y * a.Hi[4] + z * a.Hi[7]);
    const double f2 = rint(x * a.Hi[2] + y * a.Hi[5] + z * a.Hi[8]);
    x -= f0 * a.H[0] + f1 * a.H[3] + f2 * a.H[6];
    y -= f0 * a.H[1] + f1 * a.H[4] + f2 * a.H[7];
    z -= f0 * a.H[2] + f1 * a.H[5] + f2 * a.H[8];
  }
}

__device__ __forceinline__ void load_pos4(const double *pos4, int j, double &x, double &y, double &z, double &t) {
  const double2 *p = reinterpret_cast<const double2 *>(pos4) + 2 * (size_t)j;
  const double2 u = __ldg(p), v = __ldg(p + 1);
  x = u.x; y = u.y; z = v.x; t = v.y;
}

// Shared-memory prologue of a pair kernel: radial coefficients, the image-shift table s.H [27][4], then
// the slot -> packed-component map of this kernel (ints); returns the number of doubles used.
constexpr int kShiftLut = 27 * 4;
__device__ __forceinline__ int stage_coef(const PairArgs &a, double *csm, int n_kmap) {
  const int n = a.n_species * a.n_species * a.crow;        // crow is even
  for (int i = threadIdx.x; i < n; i += blockDim.x) csm[i] = a.coef[i];
  if (threadIdx.x < 27) {
    const int q = (threadIdx.x + 13) % 27;                  // code -> position in the {-1,0,1}^3 list
    const double s0 = q / 9 - 1, s1 = (q / 3) % 3 - 1, s2 = q % 3 - 1;
    double *o = csm + n + 4 * threadIdx.x;
    o[0] = s0 * a.H[0] + s1 * a.H[3] + s2 * a.H[6];
    o[1] = s0 * a.H[1] + s1 * a.H[4] + s2 * a.H[7];
    o[2] = s0 * a.H[2] + s1 * a.H[5] + s2 * a.H[8];
    o[3] = 0.0;
  }
  int *km = reinterpret_cast<int *>(csm + n + kShiftLut);
  for (int i = threadIdx.x; i < n_kmap; i += blockDim.x) km[i] = a.kmap[i];
  __syncthreads();
  return n + kShiftLut + ((n_kmap + 3) / 4) * 2;            // keep 16-byte alignment
}

}  // namespace mtpb
