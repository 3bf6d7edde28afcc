// Host-side compilation of the flat contraction table (include/mtp_b200.h) into the wave /
// item schedule the K2 kernel interprets.  BASELINE.json north_star: "a forward/adjoint
// contraction kernel with the tree in registers and shared memory" -- the table itself is an
// input of mtp_create, so any valid table (not only mtp_enumerate's) is accepted.
#include "tree.h"

#include <algorithm>

#include "mtp_b200.h"

namespace mtpb {

int tree_compile(int n_basic, int n_nodes, int n_prod, const int32_t *prod, int n_basis,
                 const int32_t *basis_node, const double *xi, int R, TreeSched &s, const char **err) {
  static const char *e_range = "contraction table: node index out of range";
  static const char *e_order = "contraction table: a node is read before its last write";
  static const char *e_big = "contraction table: more than 65535 nodes";
  if (n_nodes > 65535) { *err = e_big; return MTP_EUNSUP; }
  s = TreeSched();
  s.n_nodes = n_nodes; s.n_basic = n_basic; s.n_basis = n_basis; s.n_prod = n_prod;
  std::vector<int> depth(n_nodes, 0), last_write(n_nodes, -1), first_read(n_nodes, n_prod);
  for (int t = 0; t < n_prod; ++t) {
    const int32_t *p = prod + 4 * t;
    if (p[0] < 0 || p[0] >= n_nodes || p[1] < 0 || p[1] >= n_nodes || p[3] < n_basic || p[3] >= n_nodes) {
      *err = e_range; return MTP_EINVAL;
    }
    last_write[p[3]] = t;
    first_read[p[0]] = std::min(first_read[p[0]], t);
    first_read[p[1]] = std::min(first_read[p[1]], t);
  }
  for (int n = n_basic; n < n_nodes; ++n)
    if (last_write[n] >= 0 && first_read[n] <= last_write[n]) { *err = e_order; return MTP_EINVAL; }
  for (int a = 0; a < n_basis; ++a)
    if (basis_node[a] < 0 || basis_node[a] >= n_nodes) { *err = e_range; return MTP_EINVAL; }
  // depth: list order is a valid evaluation order, so one pass suffices
  for (int t = 0; t < n_prod; ++t) {
    const int32_t *p = prod + 4 * t;
    depth[p[3]] = std::max(depth[p[3]], 1 + std::max(depth[p[0]], depth[p[1]]));
  }
  int D = 0;
  for (int n = 0; n < n_nodes; ++n) D = std::max(D, depth[n]);
  s.depth = D;

  // ---- forward rows grouped by dst, waves by depth 1..D
  std::vector<std::vector<int>> row(n_nodes);   // op ids per dst
  for (int t = 0; t < n_prod; ++t) row[prod[4 * t + 3]].push_back(t);
  // deal the rows of one wave to R lanes: longest first, always to the least-loaded lane;
  // emit the lane-major program of the wave and return its number of steps
  struct Row { int dst; std::vector<TreeTerm> terms; };
  auto deal = [R](std::vector<Row> &rows, std::vector<TreeTerm> &prog) {
    std::stable_sort(rows.begin(), rows.end(), [](const Row &x, const Row &y) { return x.terms.size() > y.terms.size(); });
    std::vector<std::vector<TreeTerm>> lane(R);
    for (auto &row : rows) {
      int best = 0;
      for (int l = 1; l < R; ++l) if (lane[l].size() < lane[best].size()) best = l;
      for (size_t k = 0; k < row.terms.size(); ++k) {
        TreeTerm t = row.terms[k];
        t.dst = (uint16_t)row.dst;
        t.last = (k + 1 == row.terms.size());
        lane[best].push_back(t);
      }
    }
    size_t S = 0;
    for (int l = 0; l < R; ++l) S = std::max(S, lane[l].size());
    S = (S + kTreePrefetch - 1) / kTreePrefetch * kTreePrefetch;
    const size_t base = prog.size();
    prog.resize(base + S * R, TreeTerm{0, 0, 0, 0, 0.0});
    for (int l = 0; l < R; ++l)
      for (size_t k = 0; k < lane[l].size(); ++k) prog[base + k * R + l] = lane[l][k];
    return (int)S;
  };
  s.R = R;
  s.fwave.push_back(0);
  for (int w = 1; w <= D; ++w) {
    std::vector<Row> rows;
    for (int n = n_basic; n < n_nodes; ++n) {
      if (depth[n] != w || row[n].empty()) continue;
      Row r; r.dst = n;
      for (int t : row[n]) {
        const int32_t *p = prod + 4 * t;
        r.terms.push_back(TreeTerm{(uint16_t)p[0], (uint16_t)p[1], 0, 0, (double)p[2]});
      }
      rows.push_back(std::move(r));
    }
    s.fwave.push_back(s.fwave.back() + deal(rows, s.fprog));
  }
  // ---- backward rows grouped by source node, waves by depth D-1 .. 0
  std::vector<std::vector<TreeTerm>> brow(n_nodes);
  for (int t = 0; t < n_prod; ++t) {
    const int32_t *p = prod + 4 * t;
    brow[p[0]].push_back(TreeTerm{(uint16_t)p[3], (uint16_t)p[1], 0, 0, (double)p[2]});
    brow[p[1]].push_back(TreeTerm{(uint16_t)p[3], (uint16_t)p[0], 0, 0, (double)p[2]});
  }
  s.bwave.push_back(0);
  for (int w = D - 1; w >= 0; --w) {
    std::vector<Row> rows;
    for (int n = 0; n < n_nodes; ++n) {
      if (depth[n] != w || brow[n].empty()) continue;
      rows.push_back(Row{n, brow[n]});
    }
    s.bwave.push_back(s.bwave.back() + deal(rows, s.bprog));
  }
  // the kernel prefetches kTreePrefetch steps ahead: pad so that those reads stay in bounds
  for (int q = 0; q < kTreePrefetch * R; ++q) { s.fprog.push_back(TreeTerm{0, 0, 0, 0, 0.0}); s.bprog.push_back(TreeTerm{0, 0, 0, 0, 0.0}); }
  // ---- adjoint seeds: dE_i/dB_alpha = xi_alpha, summed per node in alpha order
  {
    std::vector<double> sv(n_nodes, 0.0);
    std::vector<char> has(n_nodes, 0);
    for (int a = 0; a < n_basis; ++a) { sv[basis_node[a]] += xi[a]; has[basis_node[a]] = 1; }
    for (int n = 0; n < n_nodes; ++n) if (has[n]) { s.seed_node.push_back(n); s.seed_val.push_back(sv[n]); }
  }
  return MTP_OK;
}

}  // namespace mtpb
