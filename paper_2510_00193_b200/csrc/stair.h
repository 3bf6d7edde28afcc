// Compile-time description of the moment "staircase" of a level and of the lane slicing
// used by the pair kernels (rows a2-a4 and a7 of SURVEY.md 8(a)).
//
// Level rule (BASELINE.json north_star; reading G8 in DESIGN.md): M_{mu,nu} exists when
// nu = 0 and 2+4mu <= LEV, or nu >= 1 and 4mu + 2nu <= LEV - 4.
//
// Slicing: the packed components (a,b,c) of all tensors are dealt to NS = NSB*NSC lanes per
// atom by (b mod NSB, c mod NSC).  Every lane then runs the SAME instruction stream over
// "slots" (a, i, k, mu) with b = sb + NSB*i, c = sc + NSC*k; a slot whose (mu, a, b, c)
// falls outside the staircase is computed and thrown away (kmap = -1).  This keeps the
// per-lane accumulators (<= ~75 doubles) in registers without warp divergence.
#pragma once

#ifdef __CUDACC__
#define MTP_HD __host__ __device__
#else
#define MTP_HD
#endif

namespace mtpb {

template <int LEV>
struct Stair {
  static constexpr int NMU = (LEV - 2) / 4 + 1;
  MTP_HD static constexpr int numax(int mu) {
    return (LEV - 4 - 4 * mu) >= 2 ? (LEV - 4 - 4 * mu) / 2 : 0;
  }
  static constexpr int NU0 = numax(0);
  // number of mu that carry a tensor of rank nu (numax is non-increasing in mu)
  MTP_HD static constexpr int nmu_for(int nu) {
    int n = 0;
    for (int mu = 0; mu < NMU; ++mu)
      if (nu == 0 || numax(mu) >= nu) ++n;
    return n;
  }
  MTP_HD static constexpr bool valid(int mu, int nu) {
    return mu < NMU && (nu == 0 || numax(mu) >= nu);
  }
  MTP_HD static constexpr int n_basic() {
    int n = 0;
    for (int mu = 0; mu < NMU; ++mu)
      for (int nu = 0; nu <= numax(mu); ++nu) n += (nu + 1) * (nu + 2) / 2;
    return n;
  }
};

// Slot walk shared by host (kmap construction) and device (unrolled loops).
template <int LEV, int NSB, int NSC>
struct Slices {
  using St = Stair<LEV>;
  static constexpr int NS = NSB * NSC;
  static constexpr int NU0 = St::NU0;
  // number of y-columns for a given a:  b_min = NSB*i, need a + b_min <= NU0
  MTP_HD static constexpr int ncol(int a) { return (NU0 - a) / NSB + 1; }
  // number of z-steps for column (a,i): c_min = NSC*k, need a + NSB*i + c_min <= NU0
  MTP_HD static constexpr int nstep(int a, int i) { return (NU0 - a - NSB * i) / NSC + 1; }
  MTP_HD static constexpr int nmu_at(int a, int i, int k) { return St::nmu_for(a + NSB * i + NSC * k); }
  MTP_HD static constexpr int n_slots() {
    int n = 0;
    for (int a = 0; a <= NU0; ++a)
      for (int i = 0; i < ncol(a); ++i)
        for (int k = 0; k < nstep(a, i); ++k) n += nmu_at(a, i, k);
    return n;
  }
  static constexpr int NSLOT = n_slots();
};

// Which (LEV, NSB, NSC) instantiations exist.  A table whose tensors fit inside the
// staircase of a compiled level runs on that level's kernels.
struct LevelCfg { int lev, nsb, nsc; };
static constexpr LevelCfg kLevels[] = {{10, 1, 1}, {16, 1, 2}, {20, 2, 2}, {24, 2, 4}, {28, 4, 4}};
static constexpr int kNumLevels = sizeof(kLevels) / sizeof(kLevels[0]);

}  // namespace mtpb
