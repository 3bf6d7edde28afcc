// Internal launch interface between api.cu and the kernel translation units.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <string>
#include <vector>

#include "pair_kernels_args.h"
#include "tree.h"

namespace mtpb {

void count_launch();
long long launch_count();

// ---- K2
struct TreeArgs {
  const TreeTerm *fprog; const int *fwave; int nfw;
  const TreeTerm *bprog; const int *bwave; int nbw;
  int n_fprog, n_bprog;                    // entries incl. the prefetch padding
  int prog_smem_off;                       // byte offset of the staged program in shared memory (set by launch_tree)
  const double *xi0;
  const double *adj_init;                  // [n_adj] initial adjoints (slot 0 = 1, else the node's seed)
  const double *leaf_seed;                 // [n_leaf] seeds of the elided leaves
  const int *eseed_slot; const double *eseed_val; int n_eseed;   // stored nodes that are basis functions
  const int *basis_slot;                   // [n_basis] val slot of B_alpha (schedules compiled without elision)
  const int *gseed_k; const double *gseed_val; int n_gseed;   // packed moments that are basis functions
  const int *gzero_k; int n_gzero;         // packed moments no op reads
  const double *pos4;
  const double *M; double *G; long long ldm;
  double *Ei;          // [N]
  double *B;           // [N][n_basis] or null
  int n_val, n_adj, n_basic, n_basis;
  int c0, c1;
  int want_adj;
  // sub-programs of a partitioned tree (tree_partition.cpp); all null / 0 / 1 for a whole table
  const int *mload_k;                      // [n_basic] row of M / G per local packed moment, or null = identity
  const int *cut_row, *cut_vslot, *cut_aslot; int n_cut;   // the group's cut nodes: row in S / Sbar, val slot, adj slot
  double *S;                               // [n_cut_rows][ldm] cut values out (after the forward pass), or null
  const double *Sbar;                      // [n_cut_rows][ldm] dE_i/d(cut) in (seeds of the backward pass), or null
  int g_accum;                             // 1: G[k] += (groups accumulate), 0: G[k] =
  int write_energy;                        // 0: group programs leave E_i alone
};
void tree_pick_shape(int n_val, int n_adj, long long n_atoms, int *AL, int *AR);   // AL = 0: does not fit
int tree_threads(int AL);               // CTA size used with AL atom-lanes
int tree_row_lanes(int AL);             // row-lanes R = threads / AL the schedule must be dealt for
size_t tree_smem_bytes(int n_val, int n_adj, int AL, int AR);
cudaError_t launch_tree(const TreeArgs &a, int AL, int AR, cudaStream_t st);
// K2 specialised for one schedule with NVRTC (tree_jit.cpp); null when unavailable (reason in *why)
struct TreeJit;
TreeJit *tree_jit_build(const TreeSched &sc, int AL, int AR, std::string *why);
std::vector<char> tree_jit_compile(const TreeSched &sc, int AL, int AR, std::string *why);   // host only, thread-safe
TreeJit *tree_jit_load(const std::vector<char> &cubin, int AR, int NT, std::string *why);
cudaError_t tree_jit_launch(const TreeJit *j, const TreeArgs &a, cudaStream_t st);
void tree_jit_destroy(TreeJit *j);
size_t tree_jit_smem_bytes(int n_val, int n_adj, int AR, int NT);

// ---- K1 / K3: one entry per compiled level (pair_lev*.cu)
struct PairLevel {
  int lev, nsb, nsc, nslot, p_small;
  cudaError_t (*moments)(const PairArgs &a, int P, cudaStream_t st);
  cudaError_t (*pairgrad)(const PairArgs &a, int P, int atomic, cudaStream_t st, int *grid_out);
  int (*pairgrad_grid)(int n_atoms, int P);
};
const PairLevel *pair_level(int index);   // index into kLevels

// ---- misc kernels (misc_kernels.cu)
cudaError_t launch_pack(const double *pos, const int *type, int n, double *pos4, cudaStream_t st);
cudaError_t launch_zero(double *p, long long n, cudaStream_t st);
// G[k][:] = gmap[k] >= 0 ? Sbar[gmap[k]][:] : 0  (partitioned K2, before the group programs accumulate)
// S[gmap[k]][:] = M[k][:] for the packed moments that are cut nodes themselves
cudaError_t launch_scopy(double *S, long long ldm, int n_basic, int ncol, const int *gmap, const double *M, cudaStream_t st);
cudaError_t launch_ginit(double *G, long long ldm, int n_basic, int ncol, const int *gmap, const double *Sbar,
                         cudaStream_t st);
// out[p] = idx[p] | image_code(shift[p]) << 27
cudaError_t launch_pack_pairs(const int *idx, const signed char *shift, long long nnz, int *out, cudaStream_t st);
// F_k = sum_p d[p] - d[rev[p]] over row k (warp per atom, fixed order)
cudaError_t launch_gather(const long long *off, const int *rev, const double *d4, int n, double *F, cudaStream_t st);
// out[c] = sum_i in[i*stride + c] for c < ncomp <= 8, fixed order; scratch: 256 x 8 doubles (or null)
cudaError_t launch_reduce(const double *in, long long n, int stride, int ncomp, double *out, double *scratch,
                          cudaStream_t st);
// Bsum[b] = sum_i B[i][b]  (fixed order per column)
cudaError_t launch_colsum(const double *B, long long n, int nb, double *Bsum, double *scratch, cudaStream_t st);

// ---- K5 (grade_kernel.cu)
// gamma[i] = max_k | sum_a B[i][a] Ainv[a][k] |
cudaError_t launch_grade(const double *B, const double *Ainv, long long n, int nb, double *gamma, cudaStream_t st);
// gamma_cfg = max_k | sum_a Bsum[a] Ainv[a][k] |
cudaError_t launch_grade_cfg(const double *Bsum, const double *Ainv, int nb, double *scratch, double *gamma_cfg,
                             cudaStream_t st);
// fp64 FMA throughput microbenchmark
cudaError_t launch_peak_dfma(long long iters, double *sink, double *flops_out, cudaStream_t st);

}  // namespace mtpb
