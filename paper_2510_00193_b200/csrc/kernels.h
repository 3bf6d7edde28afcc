// Internal launch interface between api.cu and the kernel translation units.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <string>
#include <vector>

#include "pair_kernels_args.h"
#include "tree.h"
#include "tree_codegen.h"

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
  const double *M; double *G; int n_rows;    // tiled [tiles][n_rows][128] (kTile); n_rows = rows of M and G
  int n_cut_rows;                          // rows of the tiled S / Sbar arrays
  double *Ei;          // [N]
  double *B;           // tiled [tiles][n_basis][128] B_alpha of the chunk (column = atom - c0), or null
  int n_val, n_adj, n_basic, n_basis;
  int c0, c1;
  int want_adj;
  // sub-programs of a partitioned tree (tree_partition.cpp); all null / 0 / 1 for a whole table
  const int *mload_k;                      // [n_basic] row of M / G per local packed moment, or null = identity
  const int *cut_row, *cut_vslot, *cut_aslot; int n_cut;   // the group's cut nodes: row in S / Sbar, val slot, adj slot
  double *S;                               // tiled [tiles][n_cut_rows][128] cut values out (after the forward pass), or null
  const double *Sbar;                      // tiled, same shape: dE_i/d(cut) in (seeds of the backward pass), or null
  int g_accum;                             // 1: G[k] += (groups accumulate), 0: G[k] =
  int write_energy;                        // 0: group programs leave E_i alone
};
void tree_pick_shape(int n_val, int n_adj, long long n_atoms, int *AL, int *AR);   // AL = 0: does not fit
int tree_threads(int AL);               // CTA size used with AL atom-lanes
int tree_row_lanes(int AL);             // row-lanes R = threads / AL the schedule must be dealt for
size_t tree_smem_bytes(int n_val, int n_adj, int AL, int AR);
cudaError_t launch_tree(const TreeArgs &a, int AL, int AR, cudaStream_t st);
// K2 specialised for one table with NVRTC (tree_codegen.cpp generates the register program, tree_jit.cpp compiles
// and launches it).  All arrays tiled (kTile); one thread per atom.
struct K2Args {
  const double *in;        // [tiles][n_io][128] inputs: M (whole table, groups) or the cut values S (top program)
  double *out;             // [tiles][n_io][128] dE_i/d(input): G or dE_i/dS
  const double *sbar;      // [tiles][n_cut][128] seeds of a group program: dE_i/dS
  double *sout;            // [tiles][n_cut][128] cut values a group program exports
  double *bt;              // [tiles][n_bt][128] B_alpha (K2_VALUES of a whole table / top program)
  double *Ei;              // [N]
  const double *xi0; const double *pos4;
  int n_io, n_cut, n_bt, c0, n;
  const double *cmx;       // constants beyond the kernel's constant bank (set by k2_jit_launch)
};
struct K2Kernel;
bool k2_jit_available(std::string *why);
void k2_shape(int n_slots, int *threads, int *ctas_per_sm);   // threads = 0: does not fit
std::string k2_source(const K2Gen &g);
std::vector<char> k2_jit_compile(const K2Gen &g, std::string *why);   // host only, thread-safe
K2Kernel *k2_jit_load(const std::vector<char> &cubin, int n_slots, const std::vector<double> &consts, std::string *why);
cudaError_t k2_jit_launch(const K2Kernel *k, const K2Args &a, cudaStream_t st);
void k2_jit_destroy(K2Kernel *k);

// ---- K1 / K3: one entry per compiled level (pair_lev*.cu)
struct PairLevel {
  int lev, nsb, nsc, nslot, p_small;
  int smem_fixed;            // shared memory of a CTA besides the radial coefficients (bytes, largest variant)
  cudaError_t (*moments)(const PairArgs &a, int P, cudaStream_t st);
  cudaError_t (*pairgrad)(const PairArgs &a, int P, int atomic, cudaStream_t st, int *grid_out);
  int (*pairgrad_grid)(int n_atoms, int P);
  // large-system kernels with the components dealt to the warps of a CTA (pair_sliced.cuh); nsl = 0: the level has none
  int nsl, nslot_s, smem_fixed_s;
  cudaError_t (*moments_s)(const PairArgs &a, cudaStream_t st);
  cudaError_t (*pairgrad_s)(const PairArgs &a, int atomic, cudaStream_t st);
  int (*pairgrad_grid_s)(int n_atoms);
  void (*kmap_s)(int n_basic, const int *basic, int *out);     // [nsl][nslot_s] slot -> packed component or -1
};
const PairLevel *pair_level(int index);   // index into kLevels

// ---- misc kernels (misc_kernels.cu)
cudaError_t launch_pack(const double *pos, const int *type, int n, double *pos4, cudaStream_t st);
cudaError_t launch_zero(double *p, long long n, cudaStream_t st);
// pack + F = 0 + virial partials = 0 + touch bitmap = 0 in one launch; E and virial sums in one (two-level: two) launch
cudaError_t launch_prologue(const double *pos, const int *type, int n, double *pos4, double *F, double *wpart, long long n_wpart,
                            unsigned *touch, cudaStream_t st);
cudaError_t launch_reduce_energy_virial(const double *Ei, long long n, double *E, const double *wpart, long long n_w, double *virial,
                                        double *scratch, cudaStream_t st);
// G[k][:] = gmap[k] >= 0 ? Sbar[gmap[k]][:] : 0  (partitioned K2, before the group programs accumulate)
// S[gmap[k]][:] = M[k][:] for the packed moments that are cut nodes themselves
cudaError_t launch_scopy(double *S, int n_cut_rows, int n_basic, int ncol, const int *gmap, const double *M, cudaStream_t st);
cudaError_t launch_ginit(double *G, int n_cut_rows, int n_basic, int ncol, const int *gmap, const double *Sbar,
                         cudaStream_t st);
// dst[row][col] (leading dimension ld) = tiled src[tiles][rows][128], or the transpose dst[col][row] (ld = row length)
cudaError_t launch_untile(const double *src, int rows, long long ncol, double *dst, long long ld, int transpose, cudaStream_t st);
// the pairs [off[c0], off[c1]) of one chunk: packed words (or plain indices when shift == null; out may be null) into
// out[p - off[c0]], at most cap; touch = bitmap of kTouchWords x 32 bits marking the blocks of 2^touch_shift(n_atoms)
// atoms that hold a neighbour of the chunk
constexpr int kTouchWords = 512;
inline int touch_shift(long long n_atoms) { int s = 6; while ((n_atoms >> s) >= kTouchWords * 32) ++s; return s; }
cudaError_t launch_pack_pairs_chunk(const long long *off, int c0, int c1, const int *idx, const signed char *shift, long long n_atoms,
                                    long long cap, int *out, int *flag, unsigned *touch, cudaStream_t st, bool touch_is_zero = false);
// the same for a list with a skin (MTP_OPT_SKIN_LIST): rows compacted to the entries within R_cut (misc_kernels.cu)
cudaError_t launch_pack_rows_live(const PairArgs &a, const int *idx, const signed char *shift, long long n_atoms, long long cap, int *out,
                                  unsigned short *korig, int *cnt, double *d4, unsigned *touch, cudaStream_t st, bool touch_is_zero = false);
// F_k -= sum over the neighbours j in the chunk of d4[rev], for every atom k of a touched block
cudaError_t launch_gather_chunk(const long long *off, const int *idx, const int *rev, const double *d4, long long d4_cap, int c0,
                                int c1, int n_atoms, const unsigned *touch, double *F, cudaStream_t st);
// out[c] = sum_i in[i*stride + c] for c < ncomp <= 8, fixed order; scratch: 256 x 8 doubles (or null)
cudaError_t launch_reduce(const double *in, long long n, int stride, int ncomp, double *out, double *scratch,
                          cudaStream_t st);
// Bsum[b] += sum_i Bt[b][i] over the tiled Bt of a chunk (fixed order per row)
cudaError_t launch_colsum(const double *Bt, long long n, int nb, double *Bsum, cudaStream_t st);

// ---- device neighbour list and velocity-Verlet (neighbor_kernels.cu)
struct NbGrid { double H[9], Hi[9]; int nc[3]; };          // box rows, inverse box, cells per lattice direction
bool nb_grid(const double *box, double r_list, long long n_atoms, NbGrid &g);
size_t nb_workspace_bytes(long long n_atoms);
cudaError_t launch_scan(const int *in, long long n, long long *out, long long *totals, cudaStream_t st);
// full CSR list (rows ordered by (j, shift)), image shifts and, when rev != null, the reverse index; info[2] = {pairs
// found, errors}; at most `capacity` pairs are written
cudaError_t launch_neighbors_build(const NbGrid &g, long long n, const double *pos, double r_list, long long capacity, long long *off,
                                   int *idx, signed char *shift, int *rev, long long *info, int accumulate, void *ws, cudaStream_t st);
// text for mtp_last_error(NULL) from entry points that take no handle (defined in api.cu)
void set_thread_error(const char *msg);
cudaError_t launch_wrap(const NbGrid &g, int n, double *pos, cudaStream_t st);
cudaError_t launch_vv(int n, double *pos, double *vel, const double *F, const int *type, const double *inv_mass, double half_dt_ftm2v,
                      double dt, int drift, cudaStream_t st);
cudaError_t launch_ke(int n, const double *vel, const int *type, const double *mass, double half_mvv2e, double *ke_i, cudaStream_t st);

// ---- K5 (grade_kernel.cu)
// gamma[i] = max_k | sum_a B[i][a] Ainv[a][k] |, B given as the tiled Bt [tiles][nb][128]
cudaError_t launch_grade(const double *Bt, const double *Ainv, long long n, int nb, double *gamma, cudaStream_t st);
// gamma_cfg = max_k | sum_a Bsum[a] Ainv[a][k] |
cudaError_t launch_max_nonneg(const double *x, long long n, double *out, cudaStream_t st);
cudaError_t launch_grade_cfg(const double *Bsum, const double *Ainv, int nb, double *scratch, double *gamma_cfg,
                             cudaStream_t st);
// fp64 FMA throughput microbenchmark
cudaError_t launch_peak_dfma(long long iters, double *sink, double *flops_out, cudaStream_t st);

}  // namespace mtpb
