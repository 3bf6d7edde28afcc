// Partition of a contraction table whose node values do not fit in shared memory for a useful
// number of atoms per CTA (lev_max >= 20: 14.6 KB per atom at level 20, 65 KB at level 24).
//
// The table is cut below its "product layer" U: the nodes written by a single op of multiplicity 1
// whose consumers are all in U as well (for mtp_enumerate's tables: the products of connected
// scalars).  The cut nodes C are the factors of U-ops outside U plus the basis nodes outside U (the
// connected scalars).  Then
//   top program      nodes C (as its inputs) + U: gives E_i, every B_alpha, and dE_i/dC;
//   group programs   the ancestors (closure) of a subset of C: forward values of those cut nodes
//                    from the moments, and -- run a second time, seeded per atom with dE_i/dC --
//                    their share of G = dE_i/dM, accumulated over the groups.
// Groups are formed greedily (largest closure first, then the cut node that adds the fewest new
// nodes) under a budget of shared-memory slots, so that every program runs with 32-64 atoms per CTA.
// The price is one extra forward pass over the group programs and the nodes shared between
// groups being evaluated once per group (x1.02 at level 20, x1.2-1.4 at level 24).
// Any classification of nodes into U is valid (U is closed under consumers by construction); it
// only changes how much work moves to the small top program.  BASELINE.json north_star: "a
// forward/adjoint contraction kernel with the tree in registers and shared memory".
#include "tree_partition.h"

#include <algorithm>
#include <set>

namespace mtpb {

namespace {
int slots_of(const std::vector<char> &in, int n_basic, int n_nodes) {
  int nb = 0, ni = 0;
  for (int n = 0; n < n_nodes; ++n) if (in[n]) (n < n_basic ? nb : ni)++;
  return nb + 2 * ni + 1;
}
}  // namespace

bool tree_partition(int n_basic, int n_nodes, int n_prod, const int32_t *prod, int n_basis, const int32_t *basis_node,
                    int budget_slots, TreePartition &out) {
  out = TreePartition();
  std::vector<std::vector<int>> ops(n_nodes), cons(n_nodes);
  for (int t = 0; t < n_prod; ++t) {
    const int32_t *p = prod + 4 * t;
    ops[p[3]].push_back(t);
    cons[p[0]].push_back(p[3]);
    cons[p[1]].push_back(p[3]);
  }
  // ---- product layer U (closed under consumers)
  std::vector<char> inU(n_nodes, 0);
  for (int n = n_basic; n < n_nodes; ++n) inU[n] = ops[n].size() == 1 && prod[4 * ops[n][0] + 2] == 1;
  for (bool changed = true; changed;) {
    changed = false;
    for (int n = n_nodes - 1; n >= n_basic; --n) {
      if (!inU[n]) continue;
      for (int c : cons[n]) if (!inU[c]) { inU[n] = 0; changed = true; break; }
    }
  }
  // ---- cut nodes
  std::vector<char> isC(n_nodes, 0);
  for (int n = n_basic; n < n_nodes; ++n)
    if (inU[n]) for (int t : ops[n]) for (int q = 0; q < 2; ++q) { const int s = prod[4 * t + q]; if (!inU[s]) isC[s] = 1; }
  for (int a = 0; a < n_basis; ++a) if (!inU[basis_node[a]]) isC[basis_node[a]] = 1;
  std::vector<int> row_of(n_nodes, -1);
  for (int n = 0; n < n_nodes; ++n) if (isC[n]) { row_of[n] = (int)out.cut_node.size(); out.cut_node.push_back(n); }
  const int nC = (int)out.cut_node.size();
  if (nC == 0) return false;
  // ---- top program: C are its packed inputs, U its intermediates
  {
    TreeTable &tt = out.top;
    std::vector<int> id(n_nodes, -1);
    for (int r = 0; r < nC; ++r) id[out.cut_node[r]] = r;
    int next = nC;
    for (int n = n_basic; n < n_nodes; ++n) if (inU[n]) id[n] = next++;
    tt.n_basic = nC; tt.n_nodes = next;
    for (int t = 0; t < n_prod; ++t) {
      const int32_t *p = prod + 4 * t;
      if (!inU[p[3]]) continue;
      tt.prod.insert(tt.prod.end(), {id[p[0]], id[p[1]], p[2], id[p[3]]});
    }
    for (int a = 0; a < n_basis; ++a) tt.basis_node.push_back(id[basis_node[a]]);
  }
  for (int r = 0; r < nC; ++r) if (out.cut_node[r] < n_basic) { out.cut_basic_row.push_back(r); out.cut_basic_k.push_back(out.cut_node[r]); }
  // ---- closures of the intermediate cut nodes (ancestors below the cut, incl. packed moments)
  std::vector<int> cuts;
  for (int n : out.cut_node) if (n >= n_basic) cuts.push_back(n);
  std::vector<std::vector<int>> clo(n_nodes);          // sorted node lists, built in table order (sources first)
  for (int n = 0; n < n_nodes; ++n) {
    if (inU[n]) continue;
    std::vector<int> c{n};
    for (int t : ops[n]) for (int q = 0; q < 2; ++q) { const auto &s = clo[prod[4 * t + q]]; c.insert(c.end(), s.begin(), s.end()); }
    std::sort(c.begin(), c.end());
    c.erase(std::unique(c.begin(), c.end()), c.end());
    clo[n] = std::move(c);
  }
  // ---- greedy grouping under the slot budget
  std::vector<char> left(n_nodes, 0);
  for (int c : cuts) left[c] = 1;
  size_t n_left = cuts.size();
  while (n_left) {
    int seed = -1;
    for (int c : cuts) if (left[c] && (seed < 0 || clo[c].size() > clo[seed].size())) seed = c;
    std::vector<char> in(n_nodes, 0);
    for (int n : clo[seed]) in[n] = 1;
    int cur_slots = slots_of(in, n_basic, n_nodes);
    // (a closure that alone exceeds the budget becomes a group of its own: whether it fits is the caller's question)
    std::vector<int> members{seed};
    left[seed] = 0; --n_left;
    while (true) {
      int best = -1; size_t best_inc = 0;
      for (int c : cuts) {
        if (!left[c]) continue;
        size_t inc = 0;
        for (int n : clo[c]) inc += !in[n];
        if (best >= 0 && inc >= best_inc) continue;
        int nb = 0, ni = 0;                                                // slots of the union
        for (int n : clo[c]) if (!in[n]) (n < n_basic ? nb : ni)++;
        if (cur_slots + nb + 2 * ni > budget_slots) continue;
        best = c; best_inc = inc;
      }
      if (best < 0) break;
      for (int n : clo[best]) if (!in[n]) { in[n] = 1; cur_slots += n < n_basic ? 1 : 2; }
      members.push_back(best);
      left[best] = 0; --n_left;
    }
    // ---- the group's table: its packed moments first (local order = ascending k), then its intermediates
    TreeGroup g;
    std::vector<int> id(n_nodes, -1);
    int next = 0;
    for (int n = 0; n < n_basic; ++n) if (in[n]) { id[n] = next++; g.basic_map.push_back(n); }
    g.table.n_basic = next;
    for (int n = n_basic; n < n_nodes; ++n) if (in[n]) id[n] = next++;
    g.table.n_nodes = next;
    for (int t = 0; t < n_prod; ++t) {
      const int32_t *p = prod + 4 * t;
      if (inU[p[3]] || !in[p[3]]) continue;
      g.table.prod.insert(g.table.prod.end(), {id[p[0]], id[p[1]], p[2], id[p[3]]});
    }
    std::sort(members.begin(), members.end());
    for (int c : members) { g.cut_local.push_back(id[c]); g.cut_row.push_back(row_of[c]); }
    if (g.table.n_basic == 0) return false;       // an intermediate always descends from packed moments
    out.groups.push_back(std::move(g));
  }
  out.used = true;
  return true;
}

}  // namespace mtpb
