// Pair kernels for the large-system regime ("thread-parallel"): K1 moments, K3 pair gradient with the
// packed components of an atom dealt to the WARPS of a CTA instead of the lanes of a warp.
//
//   CTA      32 atoms x NSL slices: lane = atom, warp = slice.  A slice is a set of columns (mu, a) -- all components
//            x^a y^b z^c of M_mu with that a -- chosen at compile time by longest-first bin packing, so the slices
//            hold the same number of components to within one small column whatever the level (the residue-class
//            slicing of pair_tiled.cuh needs one instruction stream for all lanes and wastes 19 % / 30 % / 42 % of its
//            slots at level 16 / 20 / 24).  Every warp runs its own straight-line code; 33-37 components per lane
//            keep a thread at 128 registers: 16 warps per SM instead of 8.
//   tile     TN = NSL neighbours of each of the 32 atoms, one pair per thread:
//   phase A  lanes = pairs: r_ij, Chebyshev recurrence, f_mu (and f'_mu for K3) once per pair, written to the
//            shared-memory tile laid out [k][field][atom] (conflict-free for both mappings).  Neighbour words are
//            copied two tiles ahead and position records one tile ahead with cp.async, as in pair_tiled.cuh.
//   phase B  lane = atom, warp = slice: per neighbour k the slice's share of P_mu(x, y, z) = sum G x^a y^b z^c and of
//            its gradient (K3: one two-variable Horner sweep per column, 2 FMA per component), or the slice's moment
//            accumulators (K1: 1 FMA per component + 1 per row).  K3 writes the partial (sum f' P, sum f grad P) of
//            the slice to dpart[slice][k][4][atom].
//   phase C  (K3) lanes = pairs: partials summed over the slices in fixed order, d_ij to d4 (32-byte records) or fp64
//            atomics, virial partials.
// BASELINE.json north_star rows a1-a4, a7, a8; readings G1-G7, G17.
#pragma once
#include <cuda_runtime.h>
#include "pair_kernels.cuh"
#include "pair_tiled.cuh"

#ifndef K3_UNROLL_WIDE
#define K3_UNROLL_WIDE 1
#endif
#ifndef K3_UNROLL_NARROW
#define K3_UNROLL_NARROW 4
#endif

namespace mtpb {

// ---- columns (mu, a) of a level's staircase, in (mu asc, a asc) order
template <int LEV>
struct Columns {
  using St = Stair<LEV>;
  static constexpr int NMU = St::NMU;
  MTP_HD static constexpr int count() { int n = 0; for (int mu = 0; mu < NMU; ++mu) n += St::numax(mu) + 1; return n; }
  static constexpr int NCOL = count();
  MTP_HD static constexpr int index(int mu, int a) { int n = 0; for (int m = 0; m < mu; ++m) n += St::numax(m) + 1; return n + a; }
  MTP_HD static constexpr int mu_of(int c) { int mu = 0; while (c > St::numax(mu)) { c -= St::numax(mu) + 1; ++mu; } return mu; }
  MTP_HD static constexpr int a_of(int c) { int mu = 0; while (c > St::numax(mu)) { c -= St::numax(mu) + 1; ++mu; } return c; }
  MTP_HD static constexpr int deg(int c) { return St::numax(mu_of(c)) - a_of(c); }       // inner degree: b + c <= deg
  MTP_HD static constexpr int size(int c) { return (deg(c) + 1) * (deg(c) + 2) / 2; }
};

// ---- longest-processing-time bin packing of the columns into NSL slices (compile time)
template <int LEV, int NSL>
struct Slicing {
  using C = Columns<LEV>;
  static constexpr int NCOL = C::NCOL;
  struct Table { int slice_of[NCOL]; int first[NCOL]; int load[NSL]; };
  MTP_HD static constexpr Table make() {
    Table t{};
    bool done[NCOL] = {};
    for (int s = 0; s < NSL; ++s) t.load[s] = 0;
    for (int r = 0; r < NCOL; ++r) {
      int best = -1;
      for (int c = 0; c < NCOL; ++c) if (!done[c] && (best < 0 || C::size(c) > C::size(best))) best = c;
      int s = 0;
      for (int q = 1; q < NSL; ++q) if (t.load[q] < t.load[s]) s = q;
      t.slice_of[best] = s; t.load[s] += C::size(best); done[best] = true;
    }
    int next[NSL] = {};
    for (int c = 0; c < NCOL; ++c) { t.first[c] = next[t.slice_of[c]]; next[t.slice_of[c]] += C::size(c); }
    return t;
  }
  static constexpr Table T = make();
  MTP_HD static constexpr int nslot() { int m = 0; for (int s = 0; s < NSL; ++s) m = T.load[s] > m ? T.load[s] : m; return m; }
  static constexpr int NSLOT = nslot();
  MTP_HD static constexpr bool mine(int s, int mu, int a) { return T.slice_of[C::index(mu, a)] == s; }
  MTP_HD static constexpr bool has_mu(int s, int mu) {
    for (int a = 0; a <= Stair<LEV>::numax(mu); ++a) if (mine(s, mu, a)) return true;
    return false;
  }
};

// slot of component (b, c) inside a column of inner degree n: rows b = n .. 0, inside a row c = n - b .. 0
MTP_HD constexpr int col_slot(int n, int b, int c) { return (n - b) * (n - b + 1) / 2 + (n - b - c); }

// Host: slot -> packed component of the table for every slice ([NSL][NSLOT], -1 = unused slot)
template <int LEV, int NSL>
inline void sliced_kmap(int n_basic, const int *basic, int *out) {
  using C = Columns<LEV>;
  using Sl = Slicing<LEV, NSL>;
  for (int i = 0; i < NSL * Sl::NSLOT; ++i) out[i] = -1;
  for (int k = 0; k < n_basic; ++k) {
    const int mu = basic[4 * k], a = basic[4 * k + 1], b = basic[4 * k + 2], c = basic[4 * k + 3];
    if (mu >= C::NMU || a + b + c > Stair<LEV>::numax(mu)) continue;
    const int col = C::index(mu, a);
    out[Sl::T.slice_of[col] * Sl::NSLOT + Sl::T.first[col] + col_slot(C::deg(col), b, c)] = k;
  }
}

// ---- shared-memory layout of a CTA
template <int LEV, int NSL>
struct STile {
  using St = Stair<LEV>;
  static constexpr int NMU = St::NMU, TN = NSL, NT = 32 * NSL;
  static constexpr int NF1 = 3 + NMU, NF3 = 3 + 2 * NMU;            // fields per pair: x y z f[NMU] (f'[NMU])
  static constexpr int KPAD = 16 / TN >= 1 ? 16 / TN : 1;           // k stride = NF * 32 + KPAD doubles: an 8-byte access is served
                                                                    // per half-warp, whose phase-A lanes are TN k's x 16 / TN atoms:
                                                                    // with this stride they fall on 16 different bank pairs
  static constexpr int KS1 = NF1 * 32 + KPAD, KS3 = NF3 * 32 + KPAD;
  static constexpr int TILE1 = TN * KS1, TILE3 = TN * KS3;          // doubles
  static constexpr int DKS = 4 * 32 + KPAD;                         // dpart: [slice][k] blocks of [4][32] doubles
  static constexpr int DPART = NSL * TN * DKS;
  static constexpr int STAGE = 2 * NT * 4 + (3 * NT + 1) / 2 + 32 * 4;   // two position buffers (32 B per thread), three word buffers,
                                                                         // the 32 centre-atom records (x, y, z, species)
  static constexpr int CTA1 = 2 * TILE1 + STAGE, CTA3 = 2 * TILE3 + DPART + STAGE;       // the tile is double-buffered
  // CTAs per SM the register allocation aims at while a slice has <= 40 components: K1 128 registers per thread
  // (16 warps per SM); K3 168 (12 warps): with 128 its force / virial accumulators spill (measured at config 4:
  // K1 1.53 / 1.70 ms and K3 2.97 / 2.71 ms per step with 16 / 12 warps)
  // K3's neighbour loop unrolled over a whole tile interleaves independent neighbours (what hides the DFMA latency
  // with 3 warps per scheduler), but the code of all slices has to stay in the instruction cache: level 20 / 24 with
  // 8 neighbours unrolled is 137 / 225 KB of code (no_instruction 8.5 stall cycles per issue at config 3), with
  // UNR3 neighbours per trip it fits
  static constexpr int UNR3 = TN <= 4 ? K3_UNROLL_NARROW : K3_UNROLL_WIDE;
  static constexpr int MINB1 = Slicing<LEV, NSL>::NSLOT <= 40 ? (512 / NT > 0 ? 512 / NT : 1) : 1;
  static constexpr int MINB3 = Slicing<LEV, NSL>::NSLOT <= 40 ? (384 / NT > 0 ? 384 / NT : 1) : 1;
};

// cp.async staging of one pair per thread (the scheme of pair_tiled.cuh with one slot per thread)
__device__ __forceinline__ void stage_word1(const PairArgs &a, long long beg, int n_nb, int k, int *slot) {
  if (k < n_nb && beg + k < a.idx_cap) asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((unsigned)__cvta_generic_to_shared(slot)), "l"(a.idx + beg + k));
  else *slot = -1;
}
__device__ __forceinline__ void stage_pos1(const PairArgs &a, int w, double *slot, int nt) {
  if (w != -1) {
    const unsigned s0 = (unsigned)__cvta_generic_to_shared(slot);
    const double *g = a.pos4 + 4 * (size_t)(w & kIdxMask);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s0), "l"(g));
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s0 + 16 * nt), "l"(g + 2));
  }
}

// Phase A for one pair: geometry, radial functions; fields written at stride 32 doubles (zeros when the pair does not
// contribute, so that phase B needs no predicates)
template <int NMU, bool DERIV, int NB>
__device__ __forceinline__ void stage_pair_fields(const PairArgs &a, const double *__restrict__ csm, const double *__restrict__ slut, int w,
                                                  const double *rec, int nt, double xi, double yi, double zi, int zi_s,
                                                  double rc2, double *__restrict__ out) {
  double x = 0.0, y = 0.0, z = 0.0, f[NMU], df[NMU];
#pragma unroll
  for (int m = 0; m < NMU; ++m) { f[m] = 0.0; df[m] = 0.0; }
  if (w != -1) {
    const double2 p0 = *reinterpret_cast<const double2 *>(rec), p1 = *reinterpret_cast<const double2 *>(rec + 2 * nt);
    double gx, gy, gz;
    pair_vector(a, slut, (unsigned)w >> kIdxBits, xi, yi, zi, p0.x, p0.y, p1.x, gx, gy, gz);
    const double r2 = gx * gx + gy * gy + gz * gz;
    if (r2 < rc2) {
      x = gx; y = gy; z = gz;
      const double rinv = r2 > 0.0 ? rsqrt(r2) : 0.0;
      radial<NMU, DERIV, NB>(csm + (zi_s * a.n_species + (int)p1.y) * a.crow, a.nb, r2 * rinv, a.r_min, a.r_cut, a.inv_width, f, df);
      if (DERIV) {                        // K3 needs f'_mu / r (d_ij = sum f_mu grad P_mu + (sum f'_mu P_mu) r_ij / r): folded in here
#pragma unroll
        for (int m = 0; m < NMU; ++m) df[m] *= rinv;
      }
    }
  }
  out[0] = x; out[32] = y; out[64] = z;
#pragma unroll
  for (int m = 0; m < NMU; ++m) out[(3 + m) * 32] = f[m];
  if (DERIV) {
#pragma unroll
    for (int m = 0; m < NMU; ++m) out[(3 + NMU + m) * 32] = df[m];
  }
}

// ---- phase B of K3 for one column of inner degree N: R(y, z) = sum_{b + c <= N} g[b][c] y^b z^c and its two partial
// derivatives by a nested Horner sweep (z inside, y outside): 2 FMA per component + 3 per row
template <int N>
__device__ __forceinline__ void column_eval(const double *g, double y, double z, double &R, double &Ry, double &Rz) {
  R = 0.0; Ry = 0.0; Rz = 0.0;
#pragma unroll
  for (int b = N; b >= 0; --b) {
    double qv = g[col_slot(N, b, N - b)], qz = 0.0;
#pragma unroll
    for (int c = N - b - 1; c >= 0; --c) {
      qz = (c == N - b - 1) ? qv : fma(qz, z, qv);
      qv = fma(qv, z, g[col_slot(N, b, c)]);
    }
    if (b == N) { R = qv; Rz = qz; }
    else { Ry = (b == N - 1) ? R : fma(Ry, y, R); R = fma(R, y, qv); Rz = fma(Rz, y, qz); }
  }
}

// columns (MU, A), (MU, A + 1), ... of slice S: P_mu(x, y, z) restricted to the slice and its gradient
template <int LEV, int NSL, int S, int MU, int A>
__device__ __forceinline__ void k3_cols(const double *g, const double *xp, double y, double z, double &P, double &Px,
                                        double &Py, double &Pz) {
  using St = Stair<LEV>;
  using C = Columns<LEV>;
  using Sl = Slicing<LEV, NSL>;
  if constexpr (A <= St::numax(MU)) {
    if constexpr (Sl::mine(S, MU, A)) {
      constexpr int n = St::numax(MU) - A, first = Sl::T.first[C::index(MU, A)];
      if constexpr (n == 0) {
        P = fma(xp[A], g[first], P);
        if constexpr (A > 0) Px = fma((double)A * xp[A > 0 ? A - 1 : 0], g[first], Px);
      } else {
        double R, Ry, Rz;
        column_eval<n>(g + first, y, z, R, Ry, Rz);
        P = fma(xp[A], R, P); Py = fma(xp[A], Ry, Py); Pz = fma(xp[A], Rz, Pz);
        if constexpr (A > 0) Px = fma((double)A * xp[A > 0 ? A - 1 : 0], R, Px);
      }
    }
    k3_cols<LEV, NSL, S, MU, A + 1>(g, xp, y, z, P, Px, Py, Pz);
  }
}
template <int LEV, int NSL, int S, int MU>
__device__ __forceinline__ void k3_mus(const double *g, const double *__restrict__ rec, const double *xp, double y, double z,
                                       double &rs, double &dx, double &dy, double &dz) {
  using St = Stair<LEV>;
  using Sl = Slicing<LEV, NSL>;
  if constexpr (MU < St::NMU) {
    if constexpr (Sl::has_mu(S, MU)) {
      double P = 0.0, Px = 0.0, Py = 0.0, Pz = 0.0;
      k3_cols<LEV, NSL, S, MU, 0>(g, xp, y, z, P, Px, Py, Pz);
      const double f = rec[(3 + MU) * 32], df = rec[(3 + St::NMU + MU) * 32];
      rs = fma(df, P, rs); dx = fma(f, Px, dx); dy = fma(f, Py, dy); dz = fma(f, Pz, dz);
    }
    k3_mus<LEV, NSL, S, MU + 1>(g, rec, xp, y, z, rs, dx, dy, dz);
  }
}
// one neighbour: the slice's share of sum_mu f'_mu P_mu (rs) and of sum_mu f_mu grad P_mu (dx, dy, dz)
template <int LEV, int NSL, int S>
__device__ __forceinline__ void k3_slice_step(const double *g, const double *__restrict__ rec, double &rs, double &dx, double &dy, double &dz) {
  constexpr int NU0 = Stair<LEV>::NU0;
  const double x = rec[0], y = rec[32], z = rec[64];
  double xp[NU0 + 1];
  xp[0] = 1.0;
#pragma unroll
  for (int a = 1; a <= NU0; ++a) xp[a] = xp[a - 1] * x;
  rs = 0.0; dx = 0.0; dy = 0.0; dz = 0.0;
  k3_mus<LEV, NSL, S, 0>(g, rec, xp, y, z, rs, dx, dy, dz);
}

// K1: the moment accumulators of the columns (MU, A), (MU, A + 1), ... of slice S: acc[slot] += f_mu x^a y^b z^c
template <int LEV, int NSL, int S, int MU, int A>
__device__ __forceinline__ void k1_cols(double *acc, double f, const double *xp, const double *yp, const double *zp) {
  using St = Stair<LEV>;
  using C = Columns<LEV>;
  using Sl = Slicing<LEV, NSL>;
  if constexpr (A <= St::numax(MU)) {
    if constexpr (Sl::mine(S, MU, A)) {
      constexpr int n = St::numax(MU) - A, first = Sl::T.first[C::index(MU, A)];
      const double fx = A == 0 ? f : f * xp[A];
#pragma unroll
      for (int b = n; b >= 0; --b) {
        const double m = b == 0 ? fx : fx * yp[b];
#pragma unroll
        for (int c = n - b; c >= 0; --c) {
          double &t = acc[first + col_slot(n, b, c)];
          t = c == 0 ? t + m : fma(m, zp[c], t);
        }
      }
    }
    k1_cols<LEV, NSL, S, MU, A + 1>(acc, f, xp, yp, zp);
  }
}
template <int LEV, int NSL, int S, int MU>
__device__ __forceinline__ void k1_mus(double *acc, const double *__restrict__ rec, const double *xp, const double *yp, const double *zp) {
  using St = Stair<LEV>;
  using Sl = Slicing<LEV, NSL>;
  if constexpr (MU < St::NMU) {
    if constexpr (Sl::has_mu(S, MU)) k1_cols<LEV, NSL, S, MU, 0>(acc, rec[(3 + MU) * 32], xp, yp, zp);
    k1_mus<LEV, NSL, S, MU + 1>(acc, rec, xp, yp, zp);
  }
}
template <int LEV, int NSL, int S>
__device__ __forceinline__ void k1_slice_step(double *acc, const double *__restrict__ rec) {
  constexpr int NU0 = Stair<LEV>::NU0;
  const double x = rec[0], y = rec[32], z = rec[64];
  double xp[NU0 + 1], yp[NU0 + 1], zp[NU0 + 1];
  xp[0] = 1.0; yp[0] = 1.0; zp[0] = 1.0;
#pragma unroll
  for (int a = 1; a <= NU0; ++a) { xp[a] = xp[a - 1] * x; yp[a] = yp[a - 1] * y; zp[a] = zp[a - 1] * z; }
  k1_mus<LEV, NSL, S, 0>(acc, rec, xp, yp, zp);
}

// warp-uniform dispatch to the code of this warp's slice
template <int LEV, int NSL, int S = 0>
__device__ __forceinline__ void k1_dispatch(int slice, double *acc, const double *rec) {
  if constexpr (S < NSL) {
    if (slice == S) k1_slice_step<LEV, NSL, S>(acc, rec);
    else k1_dispatch<LEV, NSL, S + 1>(slice, acc, rec);
  }
}
template <int LEV, int NSL, int S = 0>
__device__ __forceinline__ void k3_dispatch(int slice, const double *g, const double *rec, double &rs, double &dx, double &dy, double &dz) {
  if constexpr (S < NSL) {
    if (slice == S) k3_slice_step<LEV, NSL, S>(g, rec, rs, dx, dy, dz);
    else k3_dispatch<LEV, NSL, S + 1>(slice, g, rec, rs, dx, dy, dz);
  }
}

// ------------------------------------------------------------------------------ K1
template <int LEV, int NSL, int NB>
__global__ void __launch_bounds__(32 * NSL, STile<LEV, NSL>::MINB1) k_moments_s(const PairArgs a) {
  using St = Stair<LEV>;
  using Sl = Slicing<LEV, NSL>;
  using Tl = STile<LEV, NSL>;
  constexpr int NMU = St::NMU, NSLOT = Sl::NSLOT, TN = Tl::TN, NT = Tl::NT, KS = Tl::KS1;
  extern __shared__ __align__(16) double csm[];
  const int ncoef = stage_coef(a, csm, NSL * NSLOT);
  const int *kmsm = reinterpret_cast<const int *>(csm + a.n_species * a.n_species * a.crow + kShiftLut);
  const double *slut = csm + a.n_species * a.n_species * a.crow;
  double *tile = csm + ncoef;
  double *pst = tile + 2 * Tl::TILE1 + 2 * threadIdx.x;           // this thread's position slot: halves NT * 16 B apart, buffers 4 NT doubles apart
  int *wst = reinterpret_cast<int *>(tile + 2 * Tl::TILE1 + 2 * NT * 4) + threadIdx.x;   // its word slots: buffers NT ints apart
  const int lane = threadIdx.x & 31, slice = threadIdx.x >> 5;
  const int atom0 = a.c0 + blockIdx.x * 32;
  // phase A role: pair (pa, pk) = neighbour pk of the tile of atom pa
  const int pa = threadIdx.x / TN, pk = threadIdx.x % TN;
  long long beg = 0;
  int n_nb = 0;
  if (atom0 + pa < a.c1) {
    beg = a.off[atom0 + pa];
    n_nb = a.cnt ? a.cnt[atom0 + pa - a.c0] : (int)(a.off[atom0 + pa + 1] - beg);
    if (a.idx_rel) beg -= a.off[a.c0];           // the neighbour words of this chunk start at 0
  }
  // the centre atoms' records live in shared memory: phase A reads its atom's (a broadcast) instead of holding
  // x, y, z, species in registers across phase B
  double *ctr = reinterpret_cast<double *>(wst - threadIdx.x + 3 * NT + (NT & 1));
  if (threadIdx.x < 32) {
    double cx = 0, cy = 0, cz = 0, ct = 0;
    if (atom0 + threadIdx.x < a.c1) load_pos4(a.pos4, atom0 + threadIdx.x, cx, cy, cz, ct);
    ctr[4 * threadIdx.x] = cx; ctr[4 * threadIdx.x + 1] = cy; ctr[4 * threadIdx.x + 2] = cz; ctr[4 * threadIdx.x + 3] = ct;
  }
  __syncthreads();
  // phase B role: lane = atom; every warp sees the same 32 atoms, so the row-length maximum is a warp reduction
  int nb_lane = 0;
  if (atom0 + lane < a.c1) nb_lane = a.cnt ? a.cnt[atom0 + lane - a.c0] : (int)(a.off[atom0 + lane + 1] - a.off[atom0 + lane]);
  const int n_max = __reduce_max_sync(0xffffffffu, nb_lane);
  const double rc2 = a.r_cut * a.r_cut;
  double acc[NSLOT];
#pragma unroll
  for (int s = 0; s < NSLOT; ++s) acc[s] = 0.0;
  stage_word1(a, beg, n_nb, pk, wst);
  stage_word1(a, beg, n_nb, TN + pk, wst + NT);
  commit_copies();
  wait_positions();
  stage_pos1(a, wst[0], pst, NT);
  commit_copies();
  int wb = 0, pb = 0;
  // phase A of tile t0: consumes the staged word / position of this tile, stages the next ones
  auto phase_a = [&](int t0, double *dst) {
    wait_positions();                                            // this tile's position and the next tile's word have landed
    const int w = wst[NT * wb];
    const double *rec = pst + 4 * NT * pb;
    const int wn = wb == 2 ? 0 : wb + 1, wnn = wn == 2 ? 0 : wn + 1;
    stage_pos1(a, wst[NT * wn], pst + 4 * NT * (pb ^ 1), NT);
    stage_word1(a, beg, n_nb, t0 + 2 * TN + pk, wst + NT * wnn);
    commit_copies();
    wb = wn; pb ^= 1;
    const double2 c0 = *reinterpret_cast<const double2 *>(ctr + 4 * pa), c1 = *reinterpret_cast<const double2 *>(ctr + 4 * pa + 2);
    stage_pair_fields<NMU, false, NB>(a, csm, slut, w, rec, NT, c0.x, c0.y, c1.x, (int)c1.y, rc2, dst + pk * KS + pa);
  };
  if (n_max > 0) phase_a(0, tile);
  __syncthreads();
  int buf = 0;
  for (int t0 = 0; t0 < n_max; t0 += TN) {
    // phase B of this tile, then phase A of the next one into the other buffer: one barrier per tile
    const double *cur = tile + buf * Tl::TILE1;
    const int kend = min(TN, n_max - t0);
    for (int k = 0; k < kend; ++k) k1_dispatch<LEV, NSL>(slice, acc, cur + k * KS + lane);
    if (t0 + TN < n_max) phase_a(t0 + TN, tile + (buf ^ 1) * Tl::TILE1);
    buf ^= 1;
    __syncthreads();
  }
  if (atom0 + lane < a.c1) {
    const int *km = kmsm + slice * NSLOT;
    double *Mc = a.M + tiled_index(a.n_rows, 0, atom0 + lane - a.c0);
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) {
      const int k = km[s];
      if (k >= 0) Mc[k * kTile] = acc[s];
    }
  }
}

// ------------------------------------------------------------------------------ K3
template <int LEV, int NSL, bool ATOMIC, int NB>
__global__ void __launch_bounds__(32 * NSL, STile<LEV, NSL>::MINB3) k_pairgrad_s(const PairArgs a) {
  using St = Stair<LEV>;
  using Sl = Slicing<LEV, NSL>;
  using Tl = STile<LEV, NSL>;
  constexpr int NMU = St::NMU, NSLOT = Sl::NSLOT, TN = Tl::TN, NT = Tl::NT, KS = Tl::KS3, DKS = Tl::DKS;
  extern __shared__ __align__(16) double csm[];
  const int ncoef = stage_coef(a, csm, NSL * NSLOT);
  const int *kmsm = reinterpret_cast<const int *>(csm + a.n_species * a.n_species * a.crow + kShiftLut);
  const double *slut = csm + a.n_species * a.n_species * a.crow;
  double *tile = csm + ncoef;
  double *dpart = tile + 2 * Tl::TILE3;
  double *pst = dpart + Tl::DPART + 2 * threadIdx.x;
  int *wst = reinterpret_cast<int *>(dpart + Tl::DPART + 2 * NT * 4) + threadIdx.x;
  const int lane = threadIdx.x & 31, slice = threadIdx.x >> 5;
  const int atom0 = a.c0 + blockIdx.x * 32;
  const int pa = threadIdx.x / TN, pk = threadIdx.x % TN;
  long long beg = 0, dbeg = 0;
  int n_nb = 0;
  if (atom0 + pa < a.c1) {
    beg = a.off[atom0 + pa];
    n_nb = a.cnt ? a.cnt[atom0 + pa - a.c0] : (int)(a.off[atom0 + pa + 1] - beg);
    dbeg = beg - a.off[a.c0];                    // d4 holds this chunk's pairs only
    if (a.idx_rel) beg = dbeg;
  }
  double *ctr = reinterpret_cast<double *>(wst - threadIdx.x + 3 * NT + (NT & 1));      // centre-atom records, as in K1
  if (threadIdx.x < 32) {
    double cx = 0, cy = 0, cz = 0, ct = 0;
    if (atom0 + threadIdx.x < a.c1) load_pos4(a.pos4, atom0 + threadIdx.x, cx, cy, cz, ct);
    ctr[4 * threadIdx.x] = cx; ctr[4 * threadIdx.x + 1] = cy; ctr[4 * threadIdx.x + 2] = cz; ctr[4 * threadIdx.x + 3] = ct;
  }
  __syncthreads();
  int nb_lane = 0;
  double g[NSLOT];
  if (atom0 + lane < a.c1) {
    nb_lane = a.cnt ? a.cnt[atom0 + lane - a.c0] : (int)(a.off[atom0 + lane + 1] - a.off[atom0 + lane]);
    const int *km = kmsm + slice * NSLOT;
    const double *Gc = a.G + tiled_index(a.n_rows, 0, atom0 + lane - a.c0);
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) {
      const int k = km[s];
      g[s] = k >= 0 ? Gc[k * kTile] : 0.0;
    }
  } else {
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) g[s] = 0.0;
  }
  const int n_max = __reduce_max_sync(0xffffffffu, nb_lane);
  const double rc2 = a.r_cut * a.r_cut;
  double Fx = 0, Fy = 0, Fz = 0, W[6] = {0, 0, 0, 0, 0, 0};
  stage_word1(a, beg, n_nb, pk, wst);
  stage_word1(a, beg, n_nb, TN + pk, wst + NT);
  commit_copies();
  wait_positions();
  stage_pos1(a, wst[0], pst, NT);
  commit_copies();
  int wb = 0, pb = 0, w_cur = -1;
  // phase A of tile t0 (lanes = pairs): returns the neighbour word of this thread's pair
  auto phase_a = [&](int t0, double *dst) {
    wait_positions();
    const int w = wst[NT * wb];
    const double *rec = pst + 4 * NT * pb;
    const int wn = wb == 2 ? 0 : wb + 1, wnn = wn == 2 ? 0 : wn + 1;
    stage_pos1(a, wst[NT * wn], pst + 4 * NT * (pb ^ 1), NT);
    stage_word1(a, beg, n_nb, t0 + 2 * TN + pk, wst + NT * wnn);
    commit_copies();
    wb = wn; pb ^= 1;
    const double2 c0 = *reinterpret_cast<const double2 *>(ctr + 4 * pa), c1 = *reinterpret_cast<const double2 *>(ctr + 4 * pa + 2);
    stage_pair_fields<NMU, true, NB>(a, csm, slut, w, rec, NT, c0.x, c0.y, c1.x, (int)c1.y, rc2, dst + pk * KS + pa);
    return w;
  };
  if (n_max > 0) w_cur = phase_a(0, tile);
  __syncthreads();
  int buf = 0;
  for (int t0 = 0; t0 < n_max; t0 += TN) {
    const double *cur = tile + buf * Tl::TILE3;
    // ---- phase B (lane = atom, warp = slice)
    const int kend = min(TN, n_max - t0);
#pragma unroll(Tl::UNR3)
    for (int k = 0; k < kend; ++k) {
      double rs = 0.0, dx = 0.0, dy = 0.0, dz = 0.0;
      k3_dispatch<LEV, NSL>(slice, g, cur + k * KS + lane, rs, dx, dy, dz);
      double *o = dpart + (slice * TN + k) * DKS + lane;
      o[0] = rs; o[32] = dx; o[64] = dy; o[96] = dz;
    }
    __syncthreads();
    // ---- phase C of this tile and phase A of the next one (both lanes = pairs; the next tile goes to the other buffer)
    {
      const int k = t0 + pk;
      if (k < n_nb && pk < kend) {
        const double *o0 = dpart + pk * DKS + pa;
        double rs = o0[0], dx = o0[32], dy = o0[64], dz = o0[96];
#pragma unroll
        for (int s = 1; s < NSL; ++s) {                            // fixed order over the slices: bit-reproducible
          const double *o = dpart + (s * TN + pk) * DKS + pa;
          rs += o[0]; dx += o[32]; dy += o[64]; dz += o[96];
        }
        const double *r = cur + pk * KS + pa;
        const double x = r[0], y = r[32], z = r[64];
        dx = fma(rs, x, dx); dy = fma(rs, y, dy); dz = fma(rs, z, dz);      // rs = sum_mu (f'_mu / r) P_mu: phase A stored f' / r
        if (ATOMIC) {
          if (dx != 0.0 || dy != 0.0 || dz != 0.0) {
            const int j = w_cur & kIdxMask;
            atomicAdd(a.F + 3 * (size_t)j, -dx);
            atomicAdd(a.F + 3 * (size_t)j + 1, -dy);
            atomicAdd(a.F + 3 * (size_t)j + 2, -dz);
          }
          Fx += dx; Fy += dy; Fz += dz;
        } else {
          const long long kd = dbeg + (a.korig ? (int)a.korig[dbeg + k] : k);      // live rows: the record keeps its CSR position
          if (kd < a.d4_cap) {
            double2 *o = reinterpret_cast<double2 *>(a.d4) + 2 * (size_t)kd;
            o[0] = make_double2(dx, dy);
            o[1] = make_double2(dz, 0.0);
            Fx += dx; Fy += dy; Fz += dz;          // the atom's own pairs are summed here, in fixed order
          } else atomicAdd(a.flag + 1, 1);
        }
        W[0] = fma(-x, dx, W[0]); W[1] = fma(-y, dy, W[1]); W[2] = fma(-z, dz, W[2]);
        W[3] = fma(-x, dy, W[3]); W[4] = fma(-x, dz, W[4]); W[5] = fma(-y, dz, W[5]);
      }
    }
    if (t0 + TN < n_max) w_cur = phase_a(t0 + TN, tile + (buf ^ 1) * Tl::TILE3);
    buf ^= 1;
    __syncthreads();
  }
  {
#pragma unroll
    for (int o = 1; o < TN; o <<= 1) {                             // the TN threads of an atom are consecutive lanes
      Fx += __shfl_xor_sync(0xffffffffu, Fx, o);
      Fy += __shfl_xor_sync(0xffffffffu, Fy, o);
      Fz += __shfl_xor_sync(0xffffffffu, Fz, o);
    }
    if (atom0 + pa < a.c1 && pk == 0) {
      double *Fo = a.F + 3 * (size_t)(atom0 + pa);
      if (ATOMIC) { atomicAdd(Fo, Fx); atomicAdd(Fo + 1, Fy); atomicAdd(Fo + 2, Fz); }
      else { Fo[0] += Fx; Fo[1] += Fy; Fo[2] += Fz; }              // one thread per atom, chunks in stream order: deterministic
    }
  }
  // virial partial of this block, fixed reduction order (deterministic)
  __shared__ double wsm[32][6];
#pragma unroll
  for (int c = 0; c < 6; ++c) {
    double v = W[c];
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) wsm[slice][c] = v;
  }
  __syncthreads();
  if (threadIdx.x < 6) {
    double v = 0;
    for (int q = 0; q < NSL; ++q) v += wsm[q][threadIdx.x];
    a.wpart[(size_t)blockIdx.x * 8 + threadIdx.x] = v;
  }
}

}  // namespace mtpb
