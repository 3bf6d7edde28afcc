// Compiled form of the contraction table for the K2 kernel (rows a5, a6 of SURVEY.md 8(a)):
// forward rows  node[dst] = sum_t mult_t node[a_t] node[b_t]           (waves by depth)
// backward rows adj[n]   += sum_t mult_t adj[dst_t] node[other_t]     (waves by depth, deepest first)
// A row is never split (no atomics -> bit-reproducible).  The host deals the rows of a wave to
// the R row-lanes of a CTA by longest-processing-time-first and emits a lane-major "program":
// step s of a wave is the R consecutive entries prog[(wave_begin + s) * R + rl]; lane rl
// executes its entry (acc += mult * src0[a] * node[b]) and, when the entry closes a row,
// stores acc to dst.  Lanes that run out of rows get no-op entries, so all lanes of a warp
// read one contiguous, fully coalesced line per step and no per-row descriptors are needed.
#pragma once
#include <cstdint>
#include <vector>

namespace mtpb {

struct TreeTerm {      // 16 bytes, one LDG.128
  uint16_t a, b;       // fwd: the two sources; bwd: a = dst whose adjoint is read, b = other source
  uint16_t dst;        // node written when this entry closes a row
  uint16_t last;       // 1: closes a row
  double mult;         // 0 for padding entries
};

constexpr int kTreePrefetch = 4;   // entries fetched ahead per lane; steps per wave are a multiple of it

struct TreeSched {
  int n_nodes = 0, n_basic = 0, n_basis = 0, depth = 0;
  std::vector<TreeTerm> fprog, bprog;  // [steps][R]
  std::vector<int32_t> fwave, bwave;   // step offsets per wave, size n_waves + 1
  std::vector<int32_t> seed_node;      // adjoint seeds: adj[seed_node[s]] = seed_val[s] (unique nodes)
  std::vector<double> seed_val;        // = sum of xi over the basis functions that live on that node
  int R = 0;                           // row-lanes the schedule was dealt for
  long long n_prod = 0;
};

// returns 0 or a negative MTP_E* code; err receives a message
int tree_compile(int n_basic, int n_nodes, int n_prod, const int32_t *prod, int n_basis,
                 const int32_t *basis_node, const double *xi, int R, TreeSched &out, const char **err);

}  // namespace mtpb
