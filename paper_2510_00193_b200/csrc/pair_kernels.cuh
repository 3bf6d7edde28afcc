// Pair kernels: K1 (a1-a4: geometry, Chebyshev radial basis, radial functions, moment
// accumulation) and K3 (a7: pair derivative d_ij = dE_i/dr_ij from the adjoints G, plus the
// per-pair part of a8).  BASELINE.json north_star; readings G1-G7, G17, G18 in DESIGN.md.
//
// Mapping (differs from the paper's Kokkos thread-/block-parallel variants):
// an atom is owned by NS*P adjacent lanes.  NS = NSB*NSC "slice" lanes split the packed
// moment components by (b mod NSB, c mod NSC) so that every lane keeps <= ~75 fp64
// accumulators in registers and all lanes of a warp run the same instruction stream
// (stair.h); P "part" lanes split the neighbour list (the small-system / block-parallel
// regime) and are combined with xor-shuffles.  All arithmetic is on the DFMA pipe.
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

// a2 + a3: f_mu(r) = (R_cut - r)^2 sum_b c[mu][b] T_b(xi),  xi = (2r - R_min - R_cut)/(R_cut - R_min)
template <int NMU, bool DERIV>
__device__ __forceinline__ void radial(const double *__restrict__ crow, int nb, double r, double r_min,
                                       double r_cut, double *f, double *df) {
  const double sx = 2.0 / (r_cut - r_min);
  const double xi = (2.0 * r - r_min - r_cut) / (r_cut - r_min);
  double s[NMU], ds[NMU];
#pragma unroll
  for (int m = 0; m < NMU; ++m) { s[m] = 0.0; ds[m] = 0.0; }
  double tm = 1.0, t = xi, dtm = 0.0, dt = 1.0;   // T_{b}, T_{b+1} and derivatives wrt xi
  for (int b = 0; b < nb; ++b) {
#pragma unroll
    for (int m = 0; m < NMU; ++m) {
      const double c = crow[m * nb + b];
      s[m] = fma(c, tm, s[m]);
      if (DERIV) ds[m] = fma(c, dtm, ds[m]);
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

// a1: r_ij = x_j - x_i + s.H, or the minimum image when no shifts are given
__device__ __forceinline__ void pair_vector(const PairArgs &a, long long p, double xi, double yi, double zi,
                                            double xj, double yj, double zj, double &x, double &y, double &z) {
  x = xj - xi; y = yj - yi; z = zj - zi;
  if (a.shift) {
    const double s0 = a.shift[3 * p], s1 = a.shift[3 * p + 1], s2 = a.shift[3 * p + 2];
    x += s0 * a.H[0] + s1 * a.H[3] + s2 * a.H[6];
    y += s0 * a.H[1] + s1 * a.H[4] + s2 * a.H[7];
    z += s0 * a.H[2] + s1 * a.H[5] + s2 * a.H[8];
  } else if (a.minimg) {
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

__device__ __forceinline__ void stage_coef(const PairArgs &a, double *csm) {
  const int n = a.n_species * a.n_species * a.crow;
  for (int i = threadIdx.x; i < n; i += blockDim.x) csm[i] = a.coef[i];
  __syncthreads();
}

// ------------------------------------------------------------------------------ K1
template <int LEV, int NSB, int NSC, int P>
__global__ void __launch_bounds__(128) k_moments(const PairArgs a) {
  using St = Stair<LEV>;
  using Sl = Slices<LEV, NSB, NSC>;
  constexpr int NMU = St::NMU, NU0 = St::NU0, NS = Sl::NS, NSLOT = Sl::NSLOT, LPA = NS * P;
  extern __shared__ double csm[];
  stage_coef(a, csm);
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int atom = a.c0 + t / LPA;
  const int q = t % LPA, slice = q % NS, part = q / NS, sb = slice % NSB, sc = slice / NSB;
  const bool act = atom < a.c1;
  double acc[NSLOT];
#pragma unroll
  for (int s = 0; s < NSLOT; ++s) acc[s] = 0.0;
  if (act) {
    double xi, yi, zi, ti;
    load_pos4(a.pos4, atom, xi, yi, zi, ti);
    const int zi_s = (int)ti;
    const long long beg = a.off[atom], end = a.off[atom + 1];
    const double rc2 = a.r_cut * a.r_cut;
    long long p = beg + part;
    double nx = 0, ny = 0, nz = 0, nt = 0;
    if (p < end) load_pos4(a.pos4, a.idx[p], nx, ny, nz, nt);
    while (p < end) {
      const double xj = nx, yj = ny, zj = nz, tj = nt;
      const long long pn = p + P;
      if (pn < end) load_pos4(a.pos4, a.idx[pn], nx, ny, nz, nt);
      double x, y, z;
      pair_vector(a, p, xi, yi, zi, xj, yj, zj, x, y, z);
      p = pn;
      const double r2 = x * x + y * y + z * z;
      if (r2 >= rc2) continue;
      const double r = r2 * rsqrt(r2);
      double f[NMU];
      radial<NMU, false>(csm + (zi_s * a.n_species + (int)tj) * a.crow, a.nb, r, a.r_min, a.r_cut, f, nullptr);
      double ysb, zs, yN, zN, dump;
      pow_small(sb, y, ysb, dump);
      pow_small(sc, z, zs, dump);
      pow_fixed<NSB>(y, yN, dump);
      pow_fixed<NSC>(z, zN, dump);
      double xa = zs;              // x^a * z^sc
      int slot = 0;
#pragma unroll
      for (int aa = 0; aa <= NU0; ++aa) {
        double col = xa * ysb;     // x^a y^(sb + NSB i) z^sc
#pragma unroll
        for (int i = 0; i < Sl::ncol(aa); ++i) {
          double tt = col;
#pragma unroll
          for (int k = 0; k < Sl::nstep(aa, i); ++k) {
#pragma unroll
            for (int m = 0; m < Sl::nmu_at(aa, i, k); ++m) { acc[slot] = fma(f[m], tt, acc[slot]); ++slot; }
            if (k + 1 < Sl::nstep(aa, i)) tt *= zN;
          }
          if (i + 1 < Sl::ncol(aa)) col *= yN;
        }
        if (aa < NU0) xa *= x;
      }
    }
  }
  if (P > 1) {
#pragma unroll
    for (int s = 0; s < NSLOT; ++s)
#pragma unroll
      for (int o = NS; o < LPA; o <<= 1) acc[s] += __shfl_xor_sync(0xffffffffu, acc[s], o);
  }
  if (act && part == 0) {
    const int *km = a.kmap + slice * NSLOT;
    double *Mc = a.M + (atom - a.c0);
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) {
      const int k = km[s];
      if (k >= 0) Mc[(long long)k * a.ldm] = acc[s];
    }
  }
}

// ------------------------------------------------------------------------------ K3
// d_ij = sum_mu [ f'_mu P_mu rhat + f_mu grad P_mu ],  P_mu(x,y,z) = sum_{abc} G_{mu,abc} x^a y^b z^c.
// Each lane evaluates its share of P_mu and its gradient by nested Horner sweeps
// (z innermost, then y, then x); slot order (mu, a desc, i desc, k desc) -- kmapB on the host.
template <int LEV, int NSB, int NSC, int P, bool ATOMIC>
__global__ void __launch_bounds__(128) k_pairgrad(const PairArgs a) {
  using St = Stair<LEV>;
  using Sl = Slices<LEV, NSB, NSC>;
  constexpr int NMU = St::NMU, NS = Sl::NS, NSLOT = Sl::NSLOT, LPA = NS * P;
  extern __shared__ double csm[];
  stage_coef(a, csm);
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int atom = a.c0 + t / LPA;
  const int q = t % LPA, slice = q % NS, part = q / NS, sb = slice % NSB, sc = slice / NSB;
  const bool act = atom < a.c1;
  double g[NSLOT];
  double Fx = 0, Fy = 0, Fz = 0, W[6] = {0, 0, 0, 0, 0, 0};
  double xi = 0, yi = 0, zi = 0, ti = 0;
  long long beg = 0, end = 0;
  if (act) {
    const int *km = a.kmap + slice * NSLOT;
    const double *Gc = a.G + (atom - a.c0);
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) {
      const int k = km[s];
      g[s] = k >= 0 ? Gc[(long long)k * a.ldm] : 0.0;
    }
    load_pos4(a.pos4, atom, xi, yi, zi, ti);
    beg = a.off[atom]; end = a.off[atom + 1];
  } else {
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) g[s] = 0.0;
  }
  const int zi_s = (int)ti;
  const double rc2 = a.r_cut * a.r_cut;
  int nit = act ? (int)((end - beg - part + P - 1) / P) : 0;
  if (nit < 0) nit = 0;
  const int maxit = (NS > 1) ? __reduce_max_sync(0xffffffffu, nit) : nit;
  long long p = beg + part;
  double nx = 0, ny = 0, nz = 0, nt = 0;
  int jn = 0;
  if (p < end) { jn = a.idx[p]; load_pos4(a.pos4, jn, nx, ny, nz, nt); }
  for (int it = 0; it < maxit; ++it) {
    const bool inrange = it < nit;
    const double xj = nx, yj = ny, zj = nz, tj = nt;
    const int j = jn;
    const long long pc = p;
    p += P;
    if (inrange && p < end) { jn = a.idx[p]; load_pos4(a.pos4, jn, nx, ny, nz, nt); }
    double dx = 0, dy = 0, dz = 0, x = 0, y = 0, z = 0;
    bool valid = false;
    if (inrange) {
      pair_vector(a, pc, xi, yi, zi, xj, yj, zj, x, y, z);
      const double r2 = x * x + y * y + z * z;
      valid = r2 < rc2;
      if (valid) {
        const double rinv = rsqrt(r2), r = r2 * rinv;
        double f[NMU], df[NMU];
        radial<NMU, true>(csm + (zi_s * a.n_species + (int)tj) * a.crow, a.nb, r, a.r_min, a.r_cut, f, df);
        double ysb, dysb, zs, dzs, yN, dyN, zN, dzN;
        pow_small(sb, y, ysb, dysb);
        pow_small(sc, z, zs, dzs);
        pow_fixed<NSB>(y, yN, dyN);
        pow_fixed<NSC>(z, zN, dzN);
        double radial_sum = 0.0;   // sum_mu f'_mu P_mu
        int slot = 0;
#pragma unroll
        for (int m = 0; m < NMU; ++m) {
          const int NUm = St::numax(m);
          double V = 0, Vx = 0, VY = 0, Vw = 0;
#pragma unroll
          for (int aa = NUm; aa >= 0; --aa) {
            double R = 0, RY = 0, Rw = 0;
#pragma unroll
            for (int i = (NUm - aa) / NSB; i >= 0; --i) {
              double qv = 0, qw = 0;
              const int kmax = (NUm - aa - NSB * i) / NSC;
#pragma unroll
              for (int k = kmax; k >= 0; --k) {
                if (k == kmax) { qv = g[slot]; }
                else { qw = (k == kmax - 1) ? qv : fma(qw, zN, qv); qv = fma(qv, zN, g[slot]); }
                ++slot;
              }
              if (i == (NUm - aa) / NSB) { R = qv; Rw = qw; }
              else { RY = (i == (NUm - aa) / NSB - 1) ? R : fma(RY, yN, R); R = fma(R, yN, qv); Rw = fma(Rw, yN, qw); }
            }
            if (aa == NUm) { V = R; VY = RY; Vw = Rw; }
            else { Vx = (aa == NUm - 1) ? V : fma(Vx, x, V); V = fma(V, x, R); VY = fma(VY, x, RY); Vw = fma(Vw, x, Rw); }
          }
          // P = ysb zs V ; Px = ysb zs Vx ; Py = zs (dysb V + ysb dyN VY) ; Pz = ysb (dzs V + zs dzN Vw)
          const double yz = ysb * zs;
          radial_sum = fma(df[m], yz * V, radial_sum);
          dx = fma(f[m], yz * Vx, dx);
          dy = fma(f[m], zs * fma(dysb, V, ysb * dyN * VY), dy);
          dz = fma(f[m], ysb * fma(dzs, V, zs * dzN * Vw), dz);
        }
        const double rs = radial_sum * rinv;
        dx = fma(rs, x, dx); dy = fma(rs, y, dy); dz = fma(rs, z, dz);
      }
    }
    if (NS > 1) {
#pragma unroll
      for (int o = 1; o < NS; o <<= 1) {
        dx += __shfl_xor_sync(0xffffffffu, dx, o);
        dy += __shfl_xor_sync(0xffffffffu, dy, o);
        dz += __shfl_xor_sync(0xffffffffu, dz, o);
      }
    }
    if (inrange && slice == 0) {
      if (ATOMIC) {
        if (valid) {
          atomicAdd(a.F + 3 * (size_t)j, -dx);
          atomicAdd(a.F + 3 * (size_t)j + 1, -dy);
          atomicAdd(a.F + 3 * (size_t)j + 2, -dz);
        }
      } else {
        double2 *o = reinterpret_cast<double2 *>(a.d4) + 2 * (size_t)pc;
        o[0] = make_double2(dx, dy);
        o[1] = make_double2(dz, 0.0);
      }
      if (valid) {
        Fx += dx; Fy += dy; Fz += dz;
        W[0] = fma(-x, dx, W[0]); W[1] = fma(-y, dy, W[1]); W[2] = fma(-z, dz, W[2]);
        W[3] = fma(-x, dy, W[3]); W[4] = fma(-x, dz, W[4]); W[5] = fma(-y, dz, W[5]);
      }
    }
  }
  if (ATOMIC) {
    if (P > 1) {
#pragma unroll
      for (int o = NS; o < LPA; o <<= 1) {
        Fx += __shfl_xor_sync(0xffffffffu, Fx, o);
        Fy += __shfl_xor_sync(0xffffffffu, Fy, o);
        Fz += __shfl_xor_sync(0xffffffffu, Fz, o);
      }
    }
    if (act && q == 0) {
      atomicAdd(a.F + 3 * (size_t)atom, Fx);
      atomicAdd(a.F + 3 * (size_t)atom + 1, Fy);
      atomicAdd(a.F + 3 * (size_t)atom + 2, Fz);
    }
  }
  // virial partial of this block, fixed reduction order (deterministic)
  __shared__ double wsm[4][6];
#pragma unroll
  for (int c = 0; c < 6; ++c) {
    double v = (slice == 0) ? W[c] : 0.0;
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) wsm[threadIdx.x >> 5][c] = v;
  }
  __syncthreads();
  if (threadIdx.x < 6) {
    double v = 0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) v += wsm[w][threadIdx.x];
    a.wpart[(size_t)blockIdx.x * 8 + threadIdx.x] = v;
  }
}

}  // namespace mtpb
