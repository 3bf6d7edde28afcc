// Partition of a large contraction table into a small "top" program over the cut nodes and group
// programs below the cut (tree_partition.cpp explains the method).
#pragma once
#include <cstdint>
#include <vector>

namespace mtpb {

struct TreeTable {                      // a contraction table in the layout of include/mtp_b200.h
  int n_basic = 0, n_nodes = 0;
  std::vector<int32_t> prod;            // [n_prod][4]
  std::vector<int32_t> basis_node;      // top program only
  int n_prod() const { return (int)(prod.size() / 4); }
};

struct TreeGroup {
  TreeTable table;                      // local numbering: the group's packed moments first
  std::vector<int32_t> basic_map;       // [table.n_basic] row of M / G of each local packed moment
  std::vector<int32_t> cut_local;       // local node ids of the group's cut nodes ...
  std::vector<int32_t> cut_row;         // ... and their rows in the cut-value arrays S / dE/dS
};

struct TreePartition {
  bool used = false;
  std::vector<int32_t> cut_node;        // original node id of every cut row (= packed input of the top program)
  std::vector<int32_t> cut_basic_row, cut_basic_k;   // cut rows that are packed moments themselves
  TreeTable top;
  std::vector<TreeGroup> groups;
};

// false: the table has no product layer to cut at.  A cut node whose closure alone exceeds the budget gets a group
// of its own.
bool tree_partition(int n_basic, int n_nodes, int n_prod, const int32_t *prod, int n_basis, const int32_t *basis_node,
                    int budget_slots, TreePartition &out);

}  // namespace mtpb
