// Compiled form of the contraction table for the K2 kernel (rows a5, a6 of SURVEY.md 8(a)):
// forward rows  node[dst] = sum_g mult_g ( sum_{t in g} node[a_t] node[b_t] )     (waves by depth)
// backward rows adj[n]   += sum_g mult_g ( sum_{t in g} adj[dst_t] node[other_t] ) (deepest first)
// The terms of a row are grouped by multiplier so that the inner step is ONE fp64 FMA per atom and
// the multiplier is applied once per group.  A row is never split (no atomics -> bit-reproducible).
//
// Storage: a CTA owns A = AL*AR atoms; thread (rl, al) handles AR atoms of atom-lane al and is
// row-lane rl of R = threads/AL.  Shared memory holds val[slot][A] for every node some op reads
// and adj[slot][A] for the intermediate nodes some op reads; "leaf" nodes (written, never read:
// the connected scalars and products at the top of the tree) get no storage when the schedule is
// compiled with elide = true: their value goes straight into E_i, and in the backward pass their
// adjoint is the constant seed xi, folded into the group multiplier with adj slot 0 (= 1.0) as
// the first factor.
//
// Program: the host deals the rows of a wave to the R row-lanes (longest processing time first)
// and emits a lane-major program: step s of a wave is the R consecutive entries
// prog[(wave_begin + s) * R + rl].  With AL = 32 a warp is one row-lane, the entry is
// warp-uniform and all shared-memory accesses are conflict-free.  Row-lanes that run out of rows
// get no-op entries.  Runs of tiny waves (the product chains at the top of the tree) are merged
// into one wave executed in order by row-lane 0, which needs no barrier between dependent rows.
#pragma once
#include <cstdint>
#include <vector>

namespace mtpb {

struct TreeTerm {      // 16 bytes, one 128-bit load
  uint32_t a;          // bits 3..: byte offset of factor 0 (fwd: in val; bwd: in adj); bits 0..2: flags
  uint32_t b;          // bits 0..17: byte offset of factor 1 in val; bits 18..31: destination index of a
                       // row-closing entry (slot in val / adj, packed-moment k, or leaf number)
  double mult;         // multiplier of the group this entry closes
};
constexpr uint32_t kTreeGroup = 1u;    // entry closes a group: tot += mult * acc, acc = 0
constexpr uint32_t kTreeRow = 2u;      // entry closes a row: dispose of tot, tot = 0
constexpr uint32_t kTreeAlt = 4u;      // row disposal: fwd 0 = store val[slot], 1 = leaf: e += leaf_seed[idx] * tot
                                       //               bwd 0 = adj[slot] += tot, 1 = G[k] = tot (global memory)
constexpr uint32_t kTreeAcc = 1u;      // in b (bit 0), backward rows without kTreeAlt: the row is a piece of a split row and
                                       // stores its partial sum into val[slot] (a spare slot) instead of adding to adj[slot]
// val slots reserved for such partial sums: 16 .. 64, growing with the number of packed inputs
inline int tree_spare_slots(int n_basic) { const int s = n_basic / 8; return s < 16 ? 16 : (s > 64 ? 64 : s); }
constexpr uint32_t kTreeBMask = ((1u << 18) - 1u) & ~7u;   // byte offset of factor 1 inside b
constexpr int kTreeDstShift = 18;
constexpr int kTreeMaxDst = 1 << 14;

constexpr int kTreePrefetch = 4;   // entries fetched ahead per lane; steps per wave are a multiple of it

struct TreeSched {
  int n_nodes = 0, n_basic = 0, n_basis = 0, depth = 0;
  int A = 0, R = 0;                    // atoms per CTA the byte offsets were scaled for; row-lanes dealt for
  bool elide = false;
  int n_val = 0, n_adj = 0;            // shared-memory slots (adj slot 0 is the constant 1)
  std::vector<TreeTerm> fprog, bprog;  // [steps][R]
  std::vector<int32_t> fwave, bwave;   // step offsets per wave, size n_waves + 1
  std::vector<int32_t> val_slot;       // [n_nodes] slot in val or -1 (elided leaf)
  std::vector<double> adj_init;        // [n_adj] initial adjoints: 1 for slot 0, the node's seed otherwise
  std::vector<double> leaf_seed;       // [n_leaf] sum of xi over the basis functions on that leaf
  std::vector<int32_t> eseed_slot;     // stored nodes that are basis functions: E_i += eseed_val * val[slot]
  std::vector<double> eseed_val;
  std::vector<int32_t> basis_slot;     // [n_basis] val slot of B_alpha (only when !elide)
  std::vector<int32_t> gseed_k;        // packed moments that are basis functions: G[k] += gseed_val
  std::vector<double> gseed_val;
  std::vector<int32_t> gzero_k;        // packed moments no op reads: G[k] = 0
  // sub-programs of a partitioned tree (tree_partition.cpp)
  std::vector<int32_t> mload_k;        // [n_basic] row of M / G each local packed moment stands for (empty: identity)
  std::vector<int32_t> cut_val_slot, cut_adj_slot;   // storage of the cut nodes, in the caller's order
  long long n_prod = 0;
  long long fsteps = 0, bsteps = 0;    // schedule length (steps per row-lane), for the cost report
};

void tree_count_slots(int n_basic, int n_nodes, int n_prod, const int32_t *prod, bool elide, int *n_val, int *n_adj,
                      const int32_t *cut_nodes = nullptr, int n_cut = 0);
// returns 0 or a negative MTP_E* code; err receives a message.  basic_map / cut_nodes describe a sub-program of a
// partitioned tree: local packed moment n stands for row basic_map[n] of M and G, cut_nodes are its outputs.
int tree_compile(int n_basic, int n_nodes, int n_prod, const int32_t *prod, int n_basis,
                 const int32_t *basis_node, const double *xi, int A, int R, bool elide, TreeSched &out,
                 const char **err, const int32_t *basic_map = nullptr, const int32_t *cut_nodes = nullptr, int n_cut = 0);

}  // namespace mtpb
