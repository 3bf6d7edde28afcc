// Host-side compilation of the flat contraction table (include/mtp_b200.h) into the wave /
// lane program the K2 kernel interprets (tree.h).  BASELINE.json north_star: "a forward/adjoint
// contraction kernel with the tree in registers and shared memory" -- the table itself is an
// input of mtp_create, so any valid table (not only mtp_enumerate's) is accepted.
#include "tree.h"

#include <algorithm>

#include "mtp_b200.h"

namespace mtpb {

namespace {
struct RawTerm { uint32_t a, b; double mult; };   // byte offsets of the two factors; group multiplier
constexpr int kTinyWaveTerms = 16;               // a wave this small may join a single-lane chain
constexpr int kTinyChainTerms = 48;              // upper bound on a merged chain
}  // namespace

void tree_count_slots(int n_basic, int n_nodes, int n_prod, const int32_t *prod, bool elide, int *n_val, int *n_adj,
                      const int32_t *cut_nodes, int n_cut) {
  std::vector<char> is_read(n_nodes, 0);
  for (int q = 0; q < n_cut; ++q) is_read[cut_nodes[q]] = 1;      // a cut node is stored like a node some op reads
  for (int t = 0; t < n_prod; ++t)
    for (int q = 0; q < 2; ++q) { const int n = prod[4 * t + q]; if (n >= 0 && n < n_nodes) is_read[n] = 1; }
  int nv = 0, na = 1;
  for (int n = 0; n < n_nodes; ++n) {
    const bool inter = n >= n_basic;
    if (!inter || is_read[n] || !elide) ++nv;
    if (inter && is_read[n]) ++na;
  }
  *n_val = nv + (n_cut > 0 ? 0 : tree_spare_slots(n_basic)); *n_adj = na;   // (group programs do not split rows)   // room for the partial sums of split backward rows
}

int tree_compile(int n_basic, int n_nodes, int n_prod, const int32_t *prod, int n_basis,
                 const int32_t *basis_node, const double *xi, int A, int R, bool elide, TreeSched &s,
                 const char **err, const int32_t *basic_map, const int32_t *cut_nodes, int n_cut) {
  const bool group = n_cut > 0;       // sub-program of a partitioned tree (tree_partition.cpp): no constant seeds
  static const char *e_range = "contraction table: node index out of range";
  static const char *e_order = "contraction table: a node is read before its last write";
  static const char *e_mult = "contraction table: negative multiplicity";
  static const char *e_big = "contraction table: too many nodes for the 14-bit destination field";
  s = TreeSched();
  s.n_nodes = n_nodes; s.n_basic = n_basic; s.n_basis = n_basis; s.n_prod = n_prod; s.A = A; s.R = R; s.elide = elide;
  std::vector<int> depth(n_nodes, 0), last_write(n_nodes, -1), first_read(n_nodes, n_prod);
  for (int t = 0; t < n_prod; ++t) {
    const int32_t *p = prod + 4 * t;
    if (p[0] < 0 || p[0] >= n_nodes || p[1] < 0 || p[1] >= n_nodes || p[3] < n_basic || p[3] >= n_nodes) {
      *err = e_range; return MTP_EINVAL;
    }
    if (p[2] < 0) { *err = e_mult; return MTP_EINVAL; }
    last_write[p[3]] = t;
    first_read[p[0]] = std::min(first_read[p[0]], t);
    first_read[p[1]] = std::min(first_read[p[1]], t);
  }
  for (int n = n_basic; n < n_nodes; ++n)
    if (first_read[n] <= last_write[n]) { *err = e_order; return MTP_EINVAL; }   // also: read but never written
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
  // seeds dE_i/dB_alpha = xi_alpha, summed per node in alpha order
  std::vector<double> seed(n_nodes, 0.0);
  std::vector<char> seeded(n_nodes, 0);
  for (int a = 0; a < n_basis; ++a) { seed[basis_node[a]] += xi[a]; seeded[basis_node[a]] = 1; }
  // ---- storage slots.  is_read[n]: some op has n as a factor.
  std::vector<char> is_read(n_nodes, 0);
  for (int t = 0; t < n_prod; ++t) { is_read[prod[4 * t]] = 1; is_read[prod[4 * t + 1]] = 1; }
  // cut nodes of a group are its outputs: their values are exported and their adjoints come in per atom,
  // so they are stored exactly like nodes some op reads
  for (int q = 0; q < n_cut; ++q) {
    if (cut_nodes[q] < n_basic || cut_nodes[q] >= n_nodes) { *err = e_range; return MTP_EINVAL; }
    is_read[cut_nodes[q]] = 1;
  }
  s.val_slot.assign(n_nodes, -1);
  std::vector<int> adj_slot(n_nodes, -1), leaf_id(n_nodes, -1);
  int nv = 0, na = 1;                                   // adj slot 0 holds the constant 1
  for (int n = 0; n < n_nodes; ++n) {
    const bool inter = n >= n_basic;
    if (!inter || is_read[n] || !elide) s.val_slot[n] = nv++;
    if (inter && is_read[n]) adj_slot[n] = na++;
    if (inter && !is_read[n] && elide) { leaf_id[n] = (int)s.leaf_seed.size(); s.leaf_seed.push_back(seed[n]); }
  }
  s.n_val = nv; s.n_adj = na;
  if (nv > kTreeMaxDst || na > kTreeMaxDst || n_basic > kTreeMaxDst || (int)s.leaf_seed.size() > kTreeMaxDst) {
    *err = e_big; return MTP_EUNSUP;
  }
  const uint32_t row_bytes = (uint32_t)A * 8u;          // one slot = A doubles
  if ((unsigned long long)nv * row_bytes >= (1ull << kTreeDstShift)) { *err = e_big; return MTP_EUNSUP; }
  s.adj_init.assign(na, 0.0);
  s.adj_init[0] = 1.0;
  for (int n = n_basic; n < n_nodes; ++n) if (adj_slot[n] >= 0) s.adj_init[adj_slot[n]] = seed[n];
  for (int n = 0; n < n_nodes; ++n)
    if (seeded[n] && s.val_slot[n] >= 0) { s.eseed_slot.push_back(s.val_slot[n]); s.eseed_val.push_back(seed[n]); }
  if (!elide) for (int a = 0; a < n_basis; ++a) s.basis_slot.push_back(s.val_slot[basis_node[a]]);

  struct Row { uint32_t dst, alt; std::vector<RawTerm> terms; bool acc = false; };
  // Emit one wave.  `single`: all rows go to row-lane 0 in the given order (dependent chain).
  auto emit = [&](std::vector<Row> &rows, bool single, std::vector<TreeTerm> &prog) {
    if (!single)
      std::stable_sort(rows.begin(), rows.end(), [](const Row &x, const Row &y) { return x.terms.size() > y.terms.size(); });
    std::vector<std::vector<TreeTerm>> lane(R);
    for (auto &row : rows) {
      int best = 0;
      if (!single)
        for (int l = 1; l < R; ++l) if (lane[l].size() < lane[best].size()) best = l;
      std::stable_sort(row.terms.begin(), row.terms.end(), [](const RawTerm &x, const RawTerm &y) { return x.mult < y.mult; });
      for (size_t k = 0; k < row.terms.size(); ++k) {
        const RawTerm &r = row.terms[k];
        TreeTerm t;
        t.a = r.a; t.b = r.b; t.mult = r.mult;
        const bool lastk = k + 1 == row.terms.size();
        if (lastk || row.terms[k + 1].mult != r.mult) t.a |= kTreeGroup;
        if (lastk) { t.a |= kTreeRow | (row.alt ? kTreeAlt : 0u); t.b |= (row.dst << kTreeDstShift) | (row.acc ? kTreeAcc : 0u); }
        lane[best].push_back(t);
      }
    }
    size_t S = 0;
    for (int l = 0; l < R; ++l) S = std::max(S, lane[l].size());
    S = (S + kTreePrefetch - 1) / kTreePrefetch * kTreePrefetch;
    const size_t base = prog.size();
    prog.resize(base + S * R, TreeTerm{0, 0, 0.0});
    for (int l = 0; l < R; ++l)
      for (size_t k = 0; k < lane[l].size(); ++k) prog[base + k * R + l] = lane[l][k];
    return (int)S;
  };
  // Emit a sequence of waves, merging runs of tiny consecutive waves into single-lane chains.
  auto emit_all = [&](std::vector<std::vector<Row>> &waves, std::vector<TreeTerm> &prog, std::vector<int32_t> &off) {
    off.push_back(0);
    auto terms_of = [](const std::vector<Row> &w) { size_t n = 0; for (auto &r : w) n += r.terms.size(); return n; };
    for (size_t w = 0; w < waves.size();) {
      if (waves[w].empty()) { ++w; continue; }
      size_t e = w, total = 0;
      while (e < waves.size() && terms_of(waves[e]) <= (size_t)kTinyWaveTerms && total + terms_of(waves[e]) <= (size_t)kTinyChainTerms) {
        total += terms_of(waves[e]); ++e;
      }
      if (e >= w + 2) {
        std::vector<Row> chain;
        for (size_t q = w; q < e; ++q) for (auto &r : waves[q]) chain.push_back(r);
        off.push_back(off.back() + emit(chain, true, prog));
        w = e;
      } else {
        off.push_back(off.back() + emit(waves[w], false, prog));
        ++w;
      }
    }
  };

  // ---- forward rows grouped by dst, waves by depth 1..D
  {
    std::vector<std::vector<int>> ops(n_nodes);
    for (int t = 0; t < n_prod; ++t) ops[prod[4 * t + 3]].push_back(t);
    std::vector<std::vector<Row>> waves(D + 1);
    for (int n = n_basic; n < n_nodes; ++n) {
      if (ops[n].empty()) continue;
      Row r;
      if (s.val_slot[n] >= 0) { r.dst = (uint32_t)s.val_slot[n]; r.alt = 0; }
      else { r.dst = (uint32_t)leaf_id[n]; r.alt = 1; }
      for (int t : ops[n]) {
        const int32_t *p = prod + 4 * t;
        r.terms.push_back(RawTerm{(uint32_t)s.val_slot[p[0]] * row_bytes, (uint32_t)s.val_slot[p[1]] * row_bytes, (double)p[2]});
      }
      waves[depth[n]].push_back(std::move(r));
    }
    emit_all(waves, s.fprog, s.fwave);
  }
  // ---- backward rows grouped by source node, waves by depth D-1 .. 0.  The adjoint of a node no
  // op reads is its constant seed: folded into the multiplier, first factor = adj slot 0 (= 1).
  std::vector<char> has_brow(n_nodes, 0);
  {
    std::vector<Row> brow(n_nodes);
    auto add = [&](int src, int other, int dst, int m) {
      RawTerm r;
      r.b = (uint32_t)s.val_slot[other] * row_bytes;
      if (adj_slot[dst] >= 0) { r.a = (uint32_t)adj_slot[dst] * row_bytes; r.mult = (double)m; }
      else {
        if (!seeded[dst] || seed[dst] == 0.0) return;   // dead: contributes nothing to E_i
        r.a = 0; r.mult = (double)m * seed[dst];
      }
      brow[src].terms.push_back(r);
    };
    for (int t = 0; t < n_prod; ++t) {
      const int32_t *p = prod + 4 * t;
      add(p[0], p[1], p[3], p[2]);
      add(p[1], p[0], p[3], p[2]);
    }
    std::vector<std::vector<Row>> waves(D + 1);
    for (int n = 0; n < n_nodes; ++n) {
      if (brow[n].terms.empty()) continue;
      has_brow[n] = 1;
      if (n < n_basic) { brow[n].dst = (uint32_t)(basic_map ? basic_map[n] : n); brow[n].alt = 1; }
      else { brow[n].dst = (uint32_t)adj_slot[n]; brow[n].alt = 0; }
      waves[D - depth[n]].push_back(std::move(brow[n]));   // deepest sources first
    }
    // A backward row much longer than its wave's share per row-lane (the adjoint of M_{0,0} collects a term from
    // every product that contains it) would serialise the wave: its terms are dealt to several pieces that run
    // concurrently in the wave and store their partial sums in spare val slots; a short row in an extra wave
    // right after adds the partials in fixed order (first factor = adj slot 0 = 1) into the real destination.
    std::vector<std::vector<Row>> split;
    int spare = 0;
    for (auto &wave : waves) {
      size_t terms = 0;
      for (auto &r : wave) terms += r.terms.size();
      const size_t lmax = std::max<size_t>(48, (terms * 5 / 4 + R - 1) / R);
      std::vector<Row> first, combine;
      for (auto &r : wave) {
        const size_t np = (r.terms.size() + lmax - 1) / lmax;
        if (r.terms.size() <= lmax + lmax / 2 || group || spare + (int)np > tree_spare_slots(n_basic)) { first.push_back(std::move(r)); continue; }
        std::stable_sort(r.terms.begin(), r.terms.end(), [](const RawTerm &x, const RawTerm &y) { return x.mult < y.mult; });
        const size_t per = (r.terms.size() + np - 1) / np;
        Row sum; sum.dst = r.dst; sum.alt = r.alt;
        for (size_t q = 0; q < np; ++q) {
          Row piece; piece.dst = (uint32_t)(nv + spare); piece.alt = 0; piece.acc = true;   // bwd + !alt + acc: store to val
          piece.terms.assign(r.terms.begin() + q * per, r.terms.begin() + std::min(r.terms.size(), (q + 1) * per));
          first.push_back(std::move(piece));
          sum.terms.push_back(RawTerm{0u, (uint32_t)(nv + spare) * row_bytes, 1.0});
          ++spare;
        }
        combine.push_back(std::move(sum));
      }
      split.push_back(std::move(first));
      if (!combine.empty()) split.push_back(std::move(combine));
    }
    s.n_val = nv + spare;
    if ((unsigned long long)s.n_val * row_bytes >= (1ull << kTreeDstShift)) { *err = e_big; return MTP_EUNSUP; }
    emit_all(split, s.bprog, s.bwave);
  }
  s.fsteps = s.fwave.back(); s.bsteps = s.bwave.back();
  // the kernel prefetches up to 4 * kTreePrefetch steps ahead: pad so that those reads stay in bounds
  for (int q = 0; q < 4 * kTreePrefetch * R; ++q) { s.fprog.push_back(TreeTerm{0, 0, 0.0}); s.bprog.push_back(TreeTerm{0, 0, 0.0}); }
  if (!group)
    for (int k = 0; k < n_basic; ++k) {
      if (seeded[k]) { s.gseed_k.push_back(k); s.gseed_val.push_back(seed[k]); }
      if (!has_brow[k]) s.gzero_k.push_back(k);
    }
  if (basic_map) s.mload_k.assign(basic_map, basic_map + n_basic);
  for (int q = 0; q < n_cut; ++q) { s.cut_val_slot.push_back(s.val_slot[cut_nodes[q]]); s.cut_adj_slot.push_back(adj_slot[cut_nodes[q]]); }
  return MTP_OK;
}

}  // namespace mtpb
