// Instantiates K1 / K3 for one compiled level and exposes them through a PairLevel record.
#pragma once
#include "kernels.h"
#include "pair_kernels.cuh"

namespace mtpb {

template <int LEV, int NSB, int NSC, int PS>
struct PairLevelImpl {
  using Sl = Slices<LEV, NSB, NSC>;
  static int grid_for(int n_atoms, int P) {
    const long long threads = (long long)n_atoms * Sl::NS * P;
    return (int)((threads + 127) / 128);
  }
  static size_t smem(const PairArgs &a) { return sizeof(double) * a.n_species * a.n_species * a.crow; }
  static cudaError_t moments(const PairArgs &a, int P, cudaStream_t st) {
    const int n = a.c1 - a.c0;
    if (n <= 0) return cudaSuccess;
    if (P == 1) k_moments<LEV, NSB, NSC, 1><<<grid_for(n, 1), 128, smem(a), st>>>(a);
    else k_moments<LEV, NSB, NSC, PS><<<grid_for(n, PS), 128, smem(a), st>>>(a);
    count_launch();
    return cudaGetLastError();
  }
  static cudaError_t pairgrad(const PairArgs &a, int P, int atomic, cudaStream_t st, int *grid_out) {
    const int n = a.c1 - a.c0;
    if (n <= 0) { if (grid_out) *grid_out = 0; return cudaSuccess; }
    const int g = grid_for(n, P == 1 ? 1 : PS);
    if (grid_out) *grid_out = g;
    if (P == 1) {
      if (atomic) k_pairgrad<LEV, NSB, NSC, 1, true><<<g, 128, smem(a), st>>>(a);
      else k_pairgrad<LEV, NSB, NSC, 1, false><<<g, 128, smem(a), st>>>(a);
    } else {
      if (atomic) k_pairgrad<LEV, NSB, NSC, PS, true><<<g, 128, smem(a), st>>>(a);
      else k_pairgrad<LEV, NSB, NSC, PS, false><<<g, 128, smem(a), st>>>(a);
    }
    count_launch();
    return cudaGetLastError();
  }
  static int pairgrad_grid(int n_atoms, int P) { return grid_for(n_atoms, P == 1 ? 1 : PS); }
  static PairLevel record() {
    return PairLevel{LEV, NSB, NSC, Sl::NSLOT, PS, &moments, &pairgrad, &pairgrad_grid};
  }
};

}  // namespace mtpb
