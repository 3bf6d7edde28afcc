// K2 code generation (rows a5, a6 of SURVEY.md 8(a)): a contraction table is turned into a straight-line
// register program for ONE atom per thread.  BASELINE.json north_star: "a forward/adjoint contraction kernel
// with the tree in registers and shared memory".
//
//   1. rows      the ops of one destination node form a row (terms grouped by multiplier); rows that cannot reach
//                an output are dropped.
//   2. schedule  forward rows in table order; the adjoint of a row runs as soon as the adjoint of its destination
//                is complete ("eager"): for a table whose seeds are known up front (group programs, whose seeds
//                dE/dS come from the top program) a graph's intermediates die right after the graph, for a whole
//                table the products of scalars at the end of the list make it the plain reverse sweep.
//                Adjoint in scatter form: for node[d] += m node[a] node[b]:  adj[a] += (m adj[d]) node[b],
//                adj[b] += (m adj[d]) node[a]; the adjoint of an elided leaf is its constant seed xi.
//   3. registers every value (node value, adjoint, temporary) lives in one of W doubles of a register window; the
//                whole access trace is known, so replacement is Belady's (evict the value whose next use is
//                furthest).  Homes of evicted values: packed inputs -> the input array itself (read-only);
//                adjoints of packed inputs -> the output array (G / dE/dS); everything else -> a private
//                shared-memory column smem[slot][thread], slots coloured by spill lifetime.
//   4. source    the physical instruction list as CUDA source for NVRTC (tree_jit.cpp); the same list is
//                exported for the host-side emulation in the tests (mtp_k2_program).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace mtpb {

struct K2Table {                        // a contraction table and its role: whole table, top program, or group program
  int n_basic = 0, n_nodes = 0;
  std::vector<int32_t> prod;            // [n_prod][4] src0, src1, mult, dst:  node[dst] += mult * node[src0] * node[src1]
  std::vector<int32_t> in_row;          // [n_basic] row of the input / output-adjoint arrays per packed input (empty: identity)
  std::vector<int32_t> basis_node;      // whole / top: node of B_alpha
  std::vector<double> xi;               // whole / top: xi_alpha
  std::vector<int32_t> cut_node, cut_row;   // group: its output nodes and their rows in S / dE/dS
  int n_prod() const { return (int)(prod.size() / 4); }
  bool is_group() const { return !cut_node.empty(); }
};

enum K2Kind {
  K2_EF = 0,        // forward + adjoint.  whole / top: E_i and OUT[row] = dE_i/d(input);  group: seeds from SBAR, OUT[row] +=
  K2_VALUES = 1     // forward only.       whole / top: BT[alpha] = B_alpha;               group: S[cut_row] = cut values
};

// Physical instruction of the register program.  Registers are indices into the window; k indexes K2Gen::consts.
enum K2Op : int32_t {
  P_LDIN = 0,    // r[d] = IN[x]                     x = row of the input array; k = 1: reload of an evicted input
  P_LDSEED = 1,  // r[d] = SBAR[x]
  P_LDOUT = 2,   // r[d] = OUT[x]                    (reload of a spilled input adjoint, or the running sum of a group)
  P_STOUT = 3,   // OUT[x] = r[a]
  P_LDS = 4,     // r[d] = smem[x]                   x = slot
  P_STS = 5,     // smem[x] = r[a]
  P_MUL = 6,     // r[d] = r[a] * r[b]
  P_FMA = 7,     // r[d] = fma(r[a], r[b], r[c])
  P_MULK = 8,    // r[d] = K[k] * r[a]
  P_FMAK = 9,    // r[d] = fma(K[k], r[a], r[c])
  P_CONST = 10,  // r[d] = K[k]
  P_ENERGY = 11, // e = fma(K[k], r[a], e)
  P_STS_OUT = 12,// S[x] = r[a]                      (group, K2_VALUES)
  P_STB = 13,    // BT[x] = r[a]                     (whole / top, K2_VALUES)
  P_ADD = 14     // r[d] = r[a] + r[c]
};
struct K2Inst { int32_t op, d, a, b, c, k, x; };

struct K2Gen {
  std::vector<K2Inst> prog;
  std::vector<double> consts;             // values of the constants for this table's weights xi
  std::vector<int32_t> const_node, const_mult;   // what they are: mult * (sum of xi on node), node = -1: the number mult
  int n_regs = 0;        // window size W
  int n_slots = 0;       // shared-memory slots per thread
  bool writes_energy = false;
  std::string source;    // preamble of the generated kernel: constant table, K2_SLOTS, K2_ENERGY
  std::string body;      // its straight-line body (tree_jit.cpp puts both into the kernel frame)
  long long n_arith = 0, n_ldg = 0, n_stg = 0, n_lds = 0, n_sts = 0;   // per atom
};

// Range / order / multiplicity checks of a table (the ones mtp_create promises): 0 or a negative MTP_E* code.
int k2_validate(int n_basic, int n_nodes, int n_prod, const int32_t *prod, int n_basis, const int32_t *basis_node,
                const char **err);

// window: doubles of the register window; lookahead: how many instructions ahead of its use a spilled operand is
// reloaded.  Returns 0 or a negative MTP_E* code.
int k2_generate(const K2Table &t, K2Kind kind, int window, int lookahead, K2Gen &out, std::string *err);

// (re)computes g.consts from the table's weights: the program itself does not depend on them
void k2_constants(const K2Table &t, K2Gen &g);

constexpr int kK2ConstBank = 4096;      // doubles of the kernel's constant bank; further constants come from global memory
constexpr int kK2Threads = 128;         // shared-memory column stride (threads per CTA the slots are laid out for)
constexpr int kK2Window = 108;          // measured at config 4: 100 / 108 doubles -> tree 0.62 / 0.60 ms per step (255 registers, no spills)
constexpr int kK2Lookahead = 2;
constexpr int kK2SlotsTwoCtas = 110;    // <= this many slots: two 128-thread CTAs per SM; up to kK2SlotsMax: one
constexpr int kK2SlotsMax = 226;
constexpr long long kK2MaxOps = 120000;  // table ops (after partitioning) above which a table is interpreted, not specialised

}  // namespace mtpb
