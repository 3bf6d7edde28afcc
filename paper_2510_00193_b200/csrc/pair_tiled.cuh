// Tiled pair kernels (K1 moments, K3 pair gradient): each warp alternates between two lane
// mappings over a tile of 128 pairs staged in shared memory.
//
//   phase A  lanes = pairs.  A warp owns NA = 32/(NS*P) atoms whose CSR rows are contiguous; a tile
//            holds neighbours [t*TN, (t+1)*TN) of each of them (TN = 4*NS*P, NA*TN = 128), four
//            consecutive pairs per lane.  a1-a3 are done ONCE per pair here: r, Chebyshev recurrence,
//            f_mu (and f'_mu for K3); the result (x, y, z, f[, f']) goes to the warp's shared-memory
//            tile.  The packed neighbour words (index + image code) are copied two tiles ahead and the
//            32-byte position records they point to one tile ahead into per-lane shared-memory staging
//            slots with cp.async (no registers held across phase B), so phase A does not wait on L2/HBM.
//            Pairs past the end of a row or with r >= R_cut are stored as zeros, so that phase B needs
//            no predicates.
//   phase B  lanes = (atom, slice, part) as in stair.h: every lane walks the TN staged pairs of its
//            atom (parts split them) and does only the part that scales with n_basic -- monomials
//            and moment FMAs (K1) or the nested Horner sweeps over G (K3).
//   phase C  (K3) lanes = pairs again: d_ij from the tile is written as full 32-byte records to
//            d4 (or scattered with fp64 atomics), virial and own-atom force partials accumulate.
// Only __syncwarp() separates the phases; warps of a CTA drift apart, so one warp's gathers
// overlap another's FMA stream.  BASELINE.json north_star rows a1-a4, a7; readings G1-G7, G17.
#pragma once
#include <cuda_runtime.h>
#include "pair_kernels.cuh"

namespace mtpb {

template <int LEV, int NSB, int NSC, int P>
struct Tile {
  using St = Stair<LEV>;
  using Sl = Slices<LEV, NSB, NSC>;
  static constexpr int NMU = St::NMU, NS = Sl::NS, LPA = NS * P, NA = 32 / LPA, TN = 4 * LPA;
  static_assert(LPA <= 32 && 32 % LPA == 0, "lanes per atom must divide the warp");
  static constexpr int PD1 = (3 + NMU + 1) & ~1;        // doubles per staged pair, K1: x y z f[NMU]
  static constexpr int PD3 = (3 + 2 * NMU + 1) & ~1;    // K3: x y z f[NMU] f'[NMU]
  static constexpr int ROW1 = TN * PD1 + 2, ROW3 = TN * PD3 + 2;   // +16 B: rows of different atoms spread over the banks
  // staging per warp: two buffers of 128 position records (x y z species) + three of 128 neighbour words
  static constexpr int STAGE = 2 * 128 * 4 + 3 * 128 / 2;
  static constexpr int WARP1 = NA * ROW1 + STAGE;        // doubles per warp
  static constexpr int WARP3 = NA * ROW3 + 128 * 4 + STAGE;   // + d_ij of the tile (three arrays of 128)
  // CTAs per SM the register allocation aims at: small per-lane slot counts leave room for more warps
  static constexpr int MINB1 = Sl::NSLOT <= 30 ? 4 : (Sl::NSLOT <= 56 ? 3 : 2), MINB3 = Sl::NSLOT <= 56 ? 3 : 2;
};

// Asynchronous copy (cp.async) of the packed neighbour words of the four pairs a lane stages in the tile
// starting at neighbour k0 into its four staging slots; -1 (an impossible word) past the row's end.
__device__ __forceinline__ void stage_words(const PairArgs &a, long long beg, int n_nb, int k0, int *slots) {
  const unsigned s0 = (unsigned)__cvta_generic_to_shared(slots);
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    if (k0 + u < n_nb && beg + k0 + u < a.idx_cap) asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(s0 + 4 * u), "l"(a.idx + beg + k0 + u));
    else slots[u] = -1;
  }
}
// Asynchronous copy of the position records of those four neighbours into this lane's staging slots.
__device__ __forceinline__ void stage_positions(const PairArgs &a, const int4 w, double *slots) {
  const unsigned s0 = (unsigned)__cvta_generic_to_shared(slots);
  const int ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    if (ww[u] != -1) {
      const double *g = a.pos4 + 4 * (size_t)(ww[u] & kIdxMask);
      asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s0 + 1024 * u), "l"(g));            // slot (u, half, lane):
      asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s0 + 1024 * u + 512), "l"(g + 2));  // lanes 16 B apart
    }
  }
}
__device__ __forceinline__ void commit_copies() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void wait_positions() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Phase A, step 1: the pair vector of one staged pair from its position record and image code.
struct PairGeo { double x, y, z; int zj; };
__device__ __forceinline__ PairGeo load_pair(const PairArgs &a, const double *__restrict__ slut, int w, const double *rec, 
                                             double xi, double yi, double zi) {
  PairGeo g{0.0, 0.0, 0.0, -1};
  if (w != -1) {
    const double2 p0 = *reinterpret_cast<const double2 *>(rec), p1 = *reinterpret_cast<const double2 *>(rec + 64);
    pair_vector(a, slut, (unsigned)w >> kIdxBits, xi, yi, zi, p0.x, p0.y, p1.x, g.x, g.y, g.z);
    g.zj = (int)p1.y;
  }
  return g;
}
// Phase A, step 2: radial functions; writes PD doubles (zeros when the pair does not contribute).
template <int NMU, bool DERIV, int PD, int NB>
__device__ __forceinline__ void stage_pair(const PairArgs &a, const double *__restrict__ csm, const PairGeo &g, int zi_s,
                                           double rc2, double *__restrict__ out) {
  double x = 0.0, y = 0.0, z = 0.0, f[NMU], df[NMU];
#pragma unroll
  for (int m = 0; m < NMU; ++m) { f[m] = 0.0; df[m] = 0.0; }
  const double r2 = g.x * g.x + g.y * g.y + g.z * g.z;
  if (g.zj >= 0 && r2 < rc2) {
    x = g.x; y = g.y; z = g.z;
    const double r = r2 * rsqrt(r2);
    radial<NMU, DERIV, NB>(csm + (zi_s * a.n_species + g.zj) * a.crow, a.nb, r, a.r_min, a.r_cut, a.inv_width, f, df);
  }
  double2 *o = reinterpret_cast<double2 *>(out);
  double buf[PD];
  buf[0] = x; buf[1] = y; buf[2] = z;
#pragma unroll
  for (int m = 0; m < NMU; ++m) buf[3 + m] = f[m];
  if (DERIV) {
#pragma unroll
    for (int m = 0; m < NMU; ++m) buf[3 + NMU + m] = df[m];
  }
#pragma unroll
  for (int q = 3 + (DERIV ? 2 : 1) * NMU; q < PD; ++q) buf[q] = 0.0;
#pragma unroll
  for (int q = 0; q < PD / 2; ++q) o[q] = make_double2(buf[2 * q], buf[2 * q + 1]);
}

// ------------------------------------------------------------------------------ K1
template <int LEV, int NSB, int NSC, int P, int NB>
__global__ void __launch_bounds__(128, Tile<LEV, NSB, NSC, P>::MINB1) k_moments_t(const PairArgs a) {
  using St = Stair<LEV>;
  using Sl = Slices<LEV, NSB, NSC>;
  using Tl = Tile<LEV, NSB, NSC, P>;
  constexpr int NMU = St::NMU, NU0 = St::NU0, NS = Sl::NS, NSLOT = Sl::NSLOT, LPA = Tl::LPA, NA = Tl::NA, TN = Tl::TN;
  constexpr int PD = Tl::PD1, ROW = Tl::ROW1;
  extern __shared__ __align__(16) double csm[];
  const int ncoef = stage_coef(a, csm, NS * NSLOT);
  const int *kmsm = reinterpret_cast<const int *>(csm + a.n_species * a.n_species * a.crow + kShiftLut);
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  double *tile = csm + ncoef + wib * Tl::WARP1;
  const int warp = blockIdx.x * (blockDim.x >> 5) + wib;
  const int sa = lane / LPA, q = lane % LPA, slice = q % NS, part = q / NS, sb = slice % NSB, sc = slice / NSB;
  const int atom = a.c0 + warp * NA + sa;
  const bool act = atom < a.c1;
  double xi = 0, yi = 0, zi = 0, ti = 0;
  long long beg = 0;
  int n_nb = 0;
  if (act) {
    load_pos4(a.pos4, atom, xi, yi, zi, ti);
    beg = a.off[atom];
    n_nb = (int)(a.off[atom + 1] - beg);
    if (a.idx_rel) beg -= a.off[a.c0];           // the neighbour words of this chunk start at 0
  }
  const int zi_s = (int)ti;
  const double rc2 = a.r_cut * a.r_cut;
  const int n_max = __reduce_max_sync(0xffffffffu, n_nb);
  double acc[NSLOT];
#pragma unroll
  for (int s = 0; s < NSLOT; ++s) acc[s] = 0.0;
  const int ka = (4 * lane) % TN;                  // phase A: this lane stages neighbours t0 + ka .. + 3 of atom slot sa
  double *mine = tile + sa * ROW;
  const double *slut = csm + a.n_species * a.n_species * a.crow;
  double *pst = tile + NA * ROW + 2 * lane;                  // this lane's position slots: (u, half) at + 128 u + 64 half doubles
  int *wst = reinterpret_cast<int *>(tile + NA * ROW + 2 * 512) + 4 * lane;   // its four word slots (buffer 0)
  stage_words(a, beg, n_nb, ka, wst);
  stage_words(a, beg, n_nb, TN + ka, wst + 128);
  commit_copies();
  wait_positions();
  stage_positions(a, *reinterpret_cast<const int4 *>(wst), pst);
  commit_copies();
  int wb = 0, pb = 0;                                       // buffers holding the current tile's words / positions
  for (int t0 = 0; t0 < n_max; t0 += TN) {
    wait_positions();                                       // positions of this tile and words of the next have landed
    const int4 jc4 = *reinterpret_cast<const int4 *>(wst + 128 * wb);
    const int jc[4] = {jc4.x, jc4.y, jc4.z, jc4.w};
    const double *rec = pst + 512 * pb;
    const int wn = wb == 2 ? 0 : wb + 1, wnn = wn == 2 ? 0 : wn + 1;
    stage_positions(a, *reinterpret_cast<const int4 *>(wst + 128 * wn), pst + 512 * (pb ^ 1));
    stage_words(a, beg, n_nb, t0 + 2 * TN + ka, wst + 128 * wnn);
    commit_copies();
    wb = wn; pb ^= 1;
    __syncwarp();
    PairGeo geo[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) geo[u] = load_pair(a, slut, jc[u], rec + 128 * u, xi, yi, zi);
#pragma unroll
    for (int u = 0; u < 4; ++u) stage_pair<NMU, false, PD, NB>(a, csm, geo[u], zi_s, rc2, mine + (ka + u) * PD);
    __syncwarp();
    const int kend = min(TN, n_max - t0);
    for (int k = part; k < kend; k += P) {
      const double2 *src = reinterpret_cast<const double2 *>(mine + k * PD);
      double buf[PD];
#pragma unroll
      for (int w = 0; w < PD / 2; ++w) { const double2 v = src[w]; buf[2 * w] = v.x; buf[2 * w + 1] = v.y; }
      const double x = buf[0], y = buf[1], z = buf[2];
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
          for (int kk = 0; kk < Sl::nstep(aa, i); ++kk) {
#pragma unroll
            for (int m = 0; m < Sl::nmu_at(aa, i, kk); ++m) { acc[slot] = fma(buf[3 + m], tt, acc[slot]); ++slot; }
            if (kk + 1 < Sl::nstep(aa, i)) tt *= zN;
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
    const int *km = kmsm + slice * NSLOT;
    double *Mc = a.M + tiled_index(a.n_rows, 0, atom - a.c0);
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) {
      const int k = km[s];
      if (k >= 0) Mc[k * kTile] = acc[s];
    }
  }
}

// ------------------------------------------------------------------------------ K3
// d_ij = sum_mu [ f'_mu P_mu rhat + f_mu grad P_mu ],  P_mu(x,y,z) = sum_{abc} G_{mu,abc} x^a y^b z^c.
// Phase B evaluates each lane's share of P_mu and its gradient by nested Horner sweeps (z innermost,
// then y, then x); slot order (mu, a desc, i desc, k desc) -- kmapB on the host.
template <int LEV, int NSB, int NSC, int P, bool ATOMIC, int NB>
__global__ void __launch_bounds__(128, Tile<LEV, NSB, NSC, P>::MINB3) k_pairgrad_t(const PairArgs a) {
  using St = Stair<LEV>;
  using Sl = Slices<LEV, NSB, NSC>;
  using Tl = Tile<LEV, NSB, NSC, P>;
  constexpr int NMU = St::NMU, NS = Sl::NS, NSLOT = Sl::NSLOT, LPA = Tl::LPA, NA = Tl::NA, TN = Tl::TN;
  constexpr int PD = Tl::PD3, ROW = Tl::ROW3;
  extern __shared__ __align__(16) double csm[];
  const int ncoef = stage_coef(a, csm, NS * NSLOT);
  const int *kmsm = reinterpret_cast<const int *>(csm + a.n_species * a.n_species * a.crow + kShiftLut);
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  double *tile = csm + ncoef + wib * Tl::WARP3;
  double *dtile = tile + NA * ROW;                  // [128][4]
  const int warp = blockIdx.x * (blockDim.x >> 5) + wib;
  const int sa = lane / LPA, q = lane % LPA, slice = q % NS, part = q / NS, sb = slice % NSB, sc = slice / NSB;
  const int atom = a.c0 + warp * NA + sa;
  const bool act = atom < a.c1;
  double g[NSLOT];
  double xi = 0, yi = 0, zi = 0, ti = 0;
  long long beg = 0, dbeg = 0;
  int n_nb = 0;
  if (act) {
    const int *km = kmsm + slice * NSLOT;
    const double *Gc = a.G + tiled_index(a.n_rows, 0, atom - a.c0);
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) {
      const int k = km[s];
      g[s] = k >= 0 ? Gc[k * kTile] : 0.0;
    }
    load_pos4(a.pos4, atom, xi, yi, zi, ti);
    beg = a.off[atom];
    n_nb = (int)(a.off[atom + 1] - beg);
    dbeg = beg - a.off[a.c0];                    // d4 holds this chunk's pairs only
    if (a.idx_rel) beg = dbeg;
  } else {
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) g[s] = 0.0;
  }
  const int zi_s = (int)ti;
  const double rc2 = a.r_cut * a.r_cut;
  const int n_max = __reduce_max_sync(0xffffffffu, n_nb);
  double Fx = 0, Fy = 0, Fz = 0, W[6] = {0, 0, 0, 0, 0, 0};
  const int ka = (4 * lane) % TN;
  double *mine = tile + sa * ROW;
  const double *slut = csm + a.n_species * a.n_species * a.crow;
  double *pst = dtile + 128 * 4 + 2 * lane;                  // this lane's position slots: (u, half) at + 128 u + 64 half doubles
  int *wst = reinterpret_cast<int *>(dtile + 128 * 4 + 2 * 512) + 4 * lane;   // its four word slots (buffer 0)
  stage_words(a, beg, n_nb, ka, wst);
  stage_words(a, beg, n_nb, TN + ka, wst + 128);
  commit_copies();
  wait_positions();
  stage_positions(a, *reinterpret_cast<const int4 *>(wst), pst);
  commit_copies();
  int wb = 0, pb = 0;                                       // buffers holding the current tile's words / positions
  for (int t0 = 0; t0 < n_max; t0 += TN) {
    wait_positions();                                       // positions of this tile and words of the next have landed
    const int4 jc4 = *reinterpret_cast<const int4 *>(wst + 128 * wb);
    const int jc[4] = {jc4.x, jc4.y, jc4.z, jc4.w};
    const double *rec = pst + 512 * pb;
    const int wn = wb == 2 ? 0 : wb + 1, wnn = wn == 2 ? 0 : wn + 1;
    stage_positions(a, *reinterpret_cast<const int4 *>(wst + 128 * wn), pst + 512 * (pb ^ 1));
    stage_words(a, beg, n_nb, t0 + 2 * TN + ka, wst + 128 * wnn);
    commit_copies();
    wb = wn; pb ^= 1;
    __syncwarp();
    // ---- phase A
#pragma unroll 1                               // one copy of the staging code: K3 is instruction-cache sensitive (measured -8 %)
    for (int u = 0; u < 4; ++u) {
      const int wu = u == 0 ? jc4.x : (u == 1 ? jc4.y : (u == 2 ? jc4.z : jc4.w));
      const PairGeo geo = load_pair(a, slut, wu, rec + 128 * u, xi, yi, zi);
      stage_pair<NMU, true, PD, NB>(a, csm, geo, zi_s, rc2, mine + (ka + u) * PD);
    }
    __syncwarp();
    // ---- phase B
    const int kend = min(TN, n_max - t0);
    for (int k0 = 0; k0 < kend; k0 += P) {
      const int k = k0 + part;                      // < TN; slots past a row's end hold zeros
      const double2 *src = reinterpret_cast<const double2 *>(mine + k * PD);
      double buf[PD];
#pragma unroll
      for (int w = 0; w < PD / 2; ++w) { const double2 v = src[w]; buf[2 * w] = v.x; buf[2 * w + 1] = v.y; }
      const double x = buf[0], y = buf[1], z = buf[2];
      const double *f = buf + 3, *df = buf + 3 + NMU;
      double dx = 0, dy = 0, dz = 0;
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
            for (int kk = kmax; kk >= 0; --kk) {
              if (kk == kmax) { qv = g[slot]; }
              else { qw = (kk == kmax - 1) ? qv : fma(qw, zN, qv); qv = fma(qv, zN, g[slot]); }
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
      const double r2 = x * x + y * y + z * z;
      const double rs = r2 > 0.0 ? radial_sum * rsqrt(r2) : 0.0;
      dx = fma(rs, x, dx); dy = fma(rs, y, dy); dz = fma(rs, z, dz);
      if (NS > 1) {
#pragma unroll
        for (int o = 1; o < NS; o <<= 1) {
          dx += __shfl_xor_sync(0xffffffffu, dx, o);
          dy += __shfl_xor_sync(0xffffffffu, dy, o);
          dz += __shfl_xor_sync(0xffffffffu, dz, o);
        }
      }
      if (slice == 0) {                           // d of the tile: three arrays [TN][NA], conflict-free here
        dtile[k * NA + sa] = dx;
        dtile[128 + k * NA + sa] = dy;
        dtile[256 + k * NA + sa] = dz;
      }
    }
    __syncwarp();
    // ---- phase C
#pragma unroll 1
    for (int u = 0; u < 4; ++u) {
      const int kl = ka + u, k = t0 + kl;
      if (k < n_nb && kl < kend) {
        const double dx = dtile[kl * NA + sa], dy = dtile[128 + kl * NA + sa], dz = dtile[256 + kl * NA + sa];
        const double2 *xy = reinterpret_cast<const double2 *>(mine + kl * PD);
        const double2 p0 = xy[0], p1 = xy[1];
        const double x = p0.x, y = p0.y, z = p1.x;
        const long long p = dbeg + k;
        if (ATOMIC) {
          if (dx != 0.0 || dy != 0.0 || dz != 0.0) {
            const int j = (u == 0 ? jc4.x : (u == 1 ? jc4.y : (u == 2 ? jc4.z : jc4.w))) & kIdxMask;
            atomicAdd(a.F + 3 * (size_t)j, -dx);
            atomicAdd(a.F + 3 * (size_t)j + 1, -dy);
            atomicAdd(a.F + 3 * (size_t)j + 2, -dz);
          }
          Fx += dx; Fy += dy; Fz += dz;
        } else {
          if (p < a.d4_cap) {
            double2 *o = reinterpret_cast<double2 *>(a.d4) + 2 * (size_t)p;
            o[0] = make_double2(dx, dy);
            o[1] = make_double2(dz, 0.0);
            Fx += dx; Fy += dy; Fz += dz;          // the atom's own pairs are summed here, in fixed order
          } else atomicAdd(a.flag + 1, 1);
        }
        W[0] = fma(-x, dx, W[0]); W[1] = fma(-y, dy, W[1]); W[2] = fma(-z, dz, W[2]);
        W[3] = fma(-x, dy, W[3]); W[4] = fma(-x, dz, W[4]); W[5] = fma(-y, dz, W[5]);
      }
    }
  }
  {
#pragma unroll
    for (int o = 1; o < LPA; o <<= 1) {
      Fx += __shfl_xor_sync(0xffffffffu, Fx, o);
      Fy += __shfl_xor_sync(0xffffffffu, Fy, o);
      Fz += __shfl_xor_sync(0xffffffffu, Fz, o);
    }
    if (act && q == 0) {
      double *Fo = a.F + 3 * (size_t)atom;
      if (ATOMIC) { atomicAdd(Fo, Fx); atomicAdd(Fo + 1, Fy); atomicAdd(Fo + 2, Fz); }
      else { Fo[0] += Fx; Fo[1] += Fy; Fo[2] += Fz; }              // one thread per atom, chunks in stream order: deterministic
    }
  }
  // virial partial of this block, fixed reduction order (deterministic)
  __shared__ double wsm[4][6];
#pragma unroll
  for (int c = 0; c < 6; ++c) {
    double v = W[c];
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) wsm[wib][c] = v;
  }
  __syncthreads();
  if (threadIdx.x < 6) {
    double v = 0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) v += wsm[w][threadIdx.x];
    a.wpart[(size_t)blockIdx.x * 8 + threadIdx.x] = v;
  }
}

}  // namespace mtpb
