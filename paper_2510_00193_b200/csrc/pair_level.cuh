// Instantiates K1 / K3 (tiled, pair_tiled.cuh) for one compiled level and exposes them through a
// PairLevel record.  P = 1 is the large-system mapping ("thread-parallel" regime), P = PS
// splits each atom's neighbours over PS lanes (the small-system / "block-parallel" regime).
#pragma once
#include "kernels.h"
#include "pair_tiled.cuh"
#include "pair_sliced.cuh"

namespace mtpb {

// the sliced (large-system) kernels of a level; NSL = 0: none
template <int LEV, int NSL>
struct SlicedImpl {
  using Sl = Slicing<LEV, NSL>;
  using Tl = STile<LEV, NSL>;
  static size_t coef_doubles(const PairArgs &a) {
    return (size_t)(a.n_species * a.n_species * a.crow) + kShiftLut + (size_t)((NSL * Sl::NSLOT + 3) / 4) * 2;
  }
  template <class K>
  static cudaError_t prep(K kernel, size_t smem) {
    // the kernels also hold a little static shared memory: opt in well below the 48 KB default limit
    return smem > 40 * 1024 ? cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) : cudaSuccess;
  }
  static int grid(int n_atoms) { return (n_atoms + 31) / 32; }
  static cudaError_t moments(const PairArgs &a, cudaStream_t st) {
    const int n = a.c1 - a.c0;
    if (n <= 0) return cudaSuccess;
    const size_t smem = 8 * (coef_doubles(a) + (size_t)Tl::CTA1);
    cudaError_t e = a.nb == 8 ? prep(k_moments_s<LEV, NSL, 8>, smem) : prep(k_moments_s<LEV, NSL, 0>, smem);
    if (e != cudaSuccess) return e;
    if (a.nb == 8) k_moments_s<LEV, NSL, 8><<<grid(n), 32 * NSL, smem, st>>>(a);
    else k_moments_s<LEV, NSL, 0><<<grid(n), 32 * NSL, smem, st>>>(a);
    count_launch();
    return cudaGetLastError();
  }
  template <bool ATOMIC>
  static cudaError_t pairgrad_a(const PairArgs &a, int n, cudaStream_t st) {
    const size_t smem = 8 * (coef_doubles(a) + (size_t)Tl::CTA3);
    cudaError_t e = a.nb == 8 ? prep(k_pairgrad_s<LEV, NSL, ATOMIC, 8>, smem) : prep(k_pairgrad_s<LEV, NSL, ATOMIC, 0>, smem);
    if (e != cudaSuccess) return e;
    if (a.nb == 8) k_pairgrad_s<LEV, NSL, ATOMIC, 8><<<grid(n), 32 * NSL, smem, st>>>(a);
    else k_pairgrad_s<LEV, NSL, ATOMIC, 0><<<grid(n), 32 * NSL, smem, st>>>(a);
    count_launch();
    return cudaGetLastError();
  }
  static cudaError_t pairgrad(const PairArgs &a, int atomic, cudaStream_t st) {
    const int n = a.c1 - a.c0;
    if (n <= 0) return cudaSuccess;
    return atomic ? pairgrad_a<true>(a, n, st) : pairgrad_a<false>(a, n, st);
  }
  static void kmap(int n_basic, const int *basic, int *out) { sliced_kmap<LEV, NSL>(n_basic, basic, out); }
  static void fill(PairLevel &r) {
    r.nsl = NSL; r.nslot_s = Sl::NSLOT;
    r.smem_fixed_s = 8 * (kShiftLut + ((NSL * Sl::NSLOT + 3) / 4) * 2 + (Tl::CTA3 > Tl::CTA1 ? Tl::CTA3 : Tl::CTA1));
    r.moments_s = &moments; r.pairgrad_s = &pairgrad; r.pairgrad_grid_s = &grid; r.kmap_s = &kmap;
  }
};
template <int LEV>
struct SlicedImpl<LEV, 0> {
  static void fill(PairLevel &r) {
    r.nsl = 0; r.nslot_s = 0; r.smem_fixed_s = 0;
    r.moments_s = nullptr; r.pairgrad_s = nullptr; r.pairgrad_grid_s = nullptr; r.kmap_s = nullptr;
  }
};

template <int LEV, int NSB, int NSC, int PS, int NSL = 0>
struct PairLevelImpl {
  using Sl = Slices<LEV, NSB, NSC>;
  static constexpr int kWarps = 4;                      // 128 threads per CTA
  template <int P>
  static int grid_for(int n_atoms) {
    const int per_cta = Tile<LEV, NSB, NSC, P>::NA * kWarps;
    return (n_atoms + per_cta - 1) / per_cta;
  }
  // shared-memory prologue: coefficients + slot map (pair_kernels.cuh stage_coef)
  static size_t coef_doubles(const PairArgs &a) {
    return (size_t)(a.n_species * a.n_species * a.crow) + kShiftLut + (size_t)((Sl::NS * Sl::NSLOT + 3) / 4) * 2;
  }
  template <class K>
  static cudaError_t prep(K kernel, size_t smem) {
    return smem > 48 * 1024 ? cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) : cudaSuccess;
  }
  template <int P>
  static cudaError_t moments_p(const PairArgs &a, int n, cudaStream_t st) {
    const size_t smem = 8 * (coef_doubles(a) + (size_t)kWarps * Tile<LEV, NSB, NSC, P>::WARP1);
    cudaError_t e = a.nb == 8 ? prep(k_moments_t<LEV, NSB, NSC, P, 8>, smem) : prep(k_moments_t<LEV, NSB, NSC, P, 0>, smem);
    if (e != cudaSuccess) return e;
    if (a.nb == 8) k_moments_t<LEV, NSB, NSC, P, 8><<<grid_for<P>(n), 32 * kWarps, smem, st>>>(a);
    else k_moments_t<LEV, NSB, NSC, P, 0><<<grid_for<P>(n), 32 * kWarps, smem, st>>>(a);
    count_launch();
    return cudaGetLastError();
  }
  template <int P, bool ATOMIC>
  static cudaError_t pairgrad_p(const PairArgs &a, int n, cudaStream_t st) {
    const size_t smem = 8 * (coef_doubles(a) + (size_t)kWarps * Tile<LEV, NSB, NSC, P>::WARP3);
    cudaError_t e = a.nb == 8 ? prep(k_pairgrad_t<LEV, NSB, NSC, P, ATOMIC, 8>, smem) : prep(k_pairgrad_t<LEV, NSB, NSC, P, ATOMIC, 0>, smem);
    if (e != cudaSuccess) return e;
    if (a.nb == 8) k_pairgrad_t<LEV, NSB, NSC, P, ATOMIC, 8><<<grid_for<P>(n), 32 * kWarps, smem, st>>>(a);
    else k_pairgrad_t<LEV, NSB, NSC, P, ATOMIC, 0><<<grid_for<P>(n), 32 * kWarps, smem, st>>>(a);
    count_launch();
    return cudaGetLastError();
  }
  static cudaError_t moments(const PairArgs &a, int P, cudaStream_t st) {
    const int n = a.c1 - a.c0;
    if (n <= 0) return cudaSuccess;
    return P == 1 ? moments_p<1>(a, n, st) : moments_p<PS>(a, n, st);
  }
  static cudaError_t pairgrad(const PairArgs &a, int P, int atomic, cudaStream_t st, int *grid_out) {
    const int n = a.c1 - a.c0;
    if (grid_out) *grid_out = n > 0 ? pairgrad_grid(n, P) : 0;
    if (n <= 0) return cudaSuccess;
    if (P == 1) return atomic ? pairgrad_p<1, true>(a, n, st) : pairgrad_p<1, false>(a, n, st);
    return atomic ? pairgrad_p<PS, true>(a, n, st) : pairgrad_p<PS, false>(a, n, st);
  }
  static int pairgrad_grid(int n_atoms, int P) { return P == 1 ? grid_for<1>(n_atoms) : grid_for<PS>(n_atoms); }
  static constexpr int max2(int a, int b) { return a > b ? a : b; }
  static PairLevel record() {
    constexpr int tile = max2(max2(Tile<LEV, NSB, NSC, 1>::WARP1, Tile<LEV, NSB, NSC, 1>::WARP3),
                              max2(Tile<LEV, NSB, NSC, PS>::WARP1, Tile<LEV, NSB, NSC, PS>::WARP3));
    const int fixed = 8 * (kShiftLut + ((Sl::NS * Sl::NSLOT + 3) / 4) * 2 + kWarps * tile);
    PairLevel r{LEV, NSB, NSC, Sl::NSLOT, PS, fixed, &moments, &pairgrad, &pairgrad_grid, 0, 0, 0, nullptr, nullptr, nullptr, nullptr};
    SlicedImpl<LEV, NSL>::fill(r);
    return r;
  }
};

}  // namespace mtpb
