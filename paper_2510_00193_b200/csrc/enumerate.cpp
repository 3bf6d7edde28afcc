// a0: host-side basis enumerator -> packed-component contraction table.
//
// BASELINE.json north_star: "a host-side basis enumerator that emits the contraction
// table"; level rule lev(M_{mu,nu}) = 2+4mu+nu summed <= lev_max.  PAPER.md:54 only says
// the level "exponentially scales the number of basis functions"; readings G8 (which
// moments exist), G9 (what a basis function is), G11 (canonical order), G12 (plain
// Einstein sums, multinomial multiplicities for packed storage) and G22 (component
// order) are restated in DESIGN.md.  This file shares nothing with oracle/basis.py.
//
// Output table semantics (include/mtp_b200.h): node[dst] += mult * node[src0] * node[src1]
// executed in list order; nodes [0, n_basic) are the packed moment components.
#include "mtp_b200.h"

#include <algorithm>
#include <array>
#include <cstdlib>
#include <cstring>
#include <map>
#include <vector>

namespace {

using Label = std::array<int, 3>;  // lev, mu, nu  (ordered by that tuple)

struct Comp {                       // a connected scalar in canonical form
  std::vector<Label> labels;
  std::vector<int> ut;              // upper-triangular adjacency, row-major
  int level() const { int s = 0; for (auto &l : labels) s += l[0]; return s; }
  bool operator<(const Comp &o) const {
    if (labels != o.labels) return labels < o.labels;   // lexicographic, prefix first
    return ut < o.ut;
  }
  bool operator==(const Comp &o) const { return labels == o.labels && ut == o.ut; }
};

inline int ut_index(int n, int i, int j) {  // i < j
  return i * n - i * (i + 1) / 2 + (j - i - 1);
}

struct Adj {
  int n;
  int k[8][8];
};

Adj to_matrix(int n, const std::vector<int> &ut) {
  Adj a; a.n = n;
  std::memset(a.k, 0, sizeof(a.k));
  for (int i = 0; i < n; ++i)
    for (int j = i + 1; j < n; ++j) a.k[i][j] = a.k[j][i] = ut[ut_index(n, i, j)];
  return a;
}

bool connected(const Adj &a, unsigned mask) {
  if (!mask) return false;
  int first = __builtin_ctz(mask);
  unsigned seen = 1u << first, frontier = seen;
  while (frontier) {
    int u = __builtin_ctz(frontier);
    frontier &= frontier - 1;
    for (int v = 0; v < a.n; ++v)
      if ((mask >> v & 1) && !(seen >> v & 1) && a.k[u][v]) { seen |= 1u << v; frontier |= 1u << v; }
  }
  return seen == mask;
}

// Smallest adjacency tuple over vertex orders that keep `keys` sorted (vertices with equal
// key may be exchanged).  `verts` lists the vertex ids, already sorted by key.  Returns the
// minimising order in `best_order`.
template <class Key>
std::vector<int> canonical_order(const Adj &a, std::vector<int> verts, const std::vector<Key> &keys,
                                 std::vector<int> *best_ut) {
  const int n = (int)verts.size();
  std::vector<int> best_order, cur = verts;
  std::vector<int> best;
  // group boundaries
  std::vector<std::pair<int, int>> groups;
  for (int i = 0; i < n;) {
    int j = i;
    while (j < n && keys[verts[j]] == keys[verts[i]]) ++j;
    groups.push_back({i, j});
    i = j;
  }
  // iterate over the product of permutations of each group
  std::vector<int> order = verts;
  for (auto &g : groups) std::sort(order.begin() + g.first, order.begin() + g.second);
  while (true) {
    std::vector<int> ut;
    ut.reserve(n * (n - 1) / 2);
    for (int i = 0; i < n; ++i)
      for (int j = i + 1; j < n; ++j) ut.push_back(a.k[order[i]][order[j]]);
    if (best_order.empty() || ut < best) { best = ut; best_order = order; }
    // advance: next permutation of the last group that can advance
    int gi = (int)groups.size() - 1;
    for (; gi >= 0; --gi) {
      if (std::next_permutation(order.begin() + groups[gi].first, order.begin() + groups[gi].second)) break;
      // wrapped around to sorted order; carry to the previous group
    }
    if (gi < 0) break;
  }
  if (best_ut) *best_ut = best;
  return best_order;
}

// ---------------------------------------------------------------- connected scalars
void enumerate_adjacencies(const std::vector<int> &nus, std::vector<std::vector<int>> &out) {
  const int n = (int)nus.size();
  std::vector<std::pair<int, int>> pairs;
  for (int i = 0; i < n; ++i) for (int j = i + 1; j < n; ++j) pairs.push_back({i, j});
  std::vector<int> rem = nus, cur;
  struct Rec {
    const std::vector<std::pair<int, int>> &pairs; int n; std::vector<int> &rem, &cur;
    std::vector<std::vector<int>> &out;
    void go(size_t p) {
      if (p == pairs.size()) {
        for (int r : rem) if (r) return;
        out.push_back(cur);
        return;
      }
      int i = pairs[p].first, j = pairs[p].second;
      int hi = std::min(rem[i], rem[j]);
      int lo = (j == n - 1) ? rem[i] : 0;
      for (int k = lo; k <= hi; ++k) {
        rem[i] -= k; rem[j] -= k; cur.push_back(k);
        go(p + 1);
        cur.pop_back(); rem[i] += k; rem[j] += k;
      }
    }
  } rec{pairs, n, rem, cur, out};
  rec.go(0);
}

std::vector<Comp> connected_scalars(int lev_max) {
  std::vector<Comp> found;
  for (int mu = 0; 2 + 4 * mu <= lev_max; ++mu) found.push_back(Comp{{Label{2 + 4 * mu, mu, 0}}, {}});
  std::vector<Label> types;
  for (int mu = 0; 2 + 4 * mu + 1 <= lev_max; ++mu)
    for (int nu = 1; 2 + 4 * mu + nu <= lev_max; ++nu) types.push_back(Label{2 + 4 * mu + nu, mu, nu});
  std::sort(types.begin(), types.end());
  std::vector<Label> chosen;
  struct Rec {
    int lev_max; const std::vector<Label> &types; std::vector<Label> &chosen; std::vector<Comp> &found;
    void go(size_t start, int total) {
      const int n = (int)chosen.size();
      if (n >= 2 && n <= 7) {
        std::vector<int> nus; int s = 0, mx = 0;
        for (auto &l : chosen) { nus.push_back(l[2]); s += l[2]; mx = std::max(mx, l[2]); }
        if (s % 2 == 0 && 2 * mx <= s && s >= 2 * (n - 1)) {
          std::vector<std::vector<int>> adjs;
          enumerate_adjacencies(nus, adjs);
          std::vector<int> verts(n);
          for (int i = 0; i < n; ++i) verts[i] = i;
          for (auto &ut : adjs) {
            Adj a = to_matrix(n, ut);
            if (!connected(a, (1u << n) - 1)) continue;
            std::vector<int> cut;
            canonical_order<Label>(a, verts, chosen, &cut);
            found.push_back(Comp{chosen, cut});
          }
        }
      }
      for (size_t t = start; t < types.size(); ++t)
        if (total + types[t][0] <= lev_max) {
          chosen.push_back(types[t]);
          go(t, total + types[t][0]);
          chosen.pop_back();
        }
    }
  } rec{lev_max, types, chosen, found};
  rec.go(0, 0);
  std::sort(found.begin(), found.end());
  found.erase(std::unique(found.begin(), found.end()), found.end());
  return found;
}

struct Func {
  int level;
  std::vector<int> comps;  // ranks into the sorted connected-scalar list, ascending
  bool operator<(const Func &o) const {
    if (level != o.level) return level < o.level;
    if (comps.size() != o.comps.size()) return comps.size() < o.comps.size();
    return comps < o.comps;
  }
};

std::vector<Func> basis_functions(int lev_max, const std::vector<Comp> &comps) {
  std::vector<int> levs;
  for (auto &c : comps) levs.push_back(c.level());
  std::vector<Func> out;
  std::vector<int> chosen;
  struct Rec {
    int lev_max; const std::vector<int> &levs; std::vector<int> &chosen; std::vector<Func> &out;
    void go(size_t start, int total) {
      if (!chosen.empty()) out.push_back(Func{total, chosen});
      for (size_t t = start; t < levs.size(); ++t)
        if (total + levs[t] <= lev_max) {
          chosen.push_back((int)t);
          go(t, total + levs[t]);
          chosen.pop_back();
        }
    }
  } rec{lev_max, levs, chosen, out};
  rec.go(0, 0);
  std::sort(out.begin(), out.end());
  return out;
}

// ---------------------------------------------------------------- contraction planner
inline int ncomp(int o) { return (o + 1) * (o + 2) / 2; }
// G22: (a,b,c) with a descending, then b descending: index = t(t+1)/2 + c, t = o - a
inline int packed_index(int a, int b, int c) { (void)b; int t = b + c; return t * (t + 1) / 2 + c; }

struct Exp3 { int a, b, c; };

void list_exponents(int o, std::vector<Exp3> &out) {
  out.clear();
  for (int a = o; a >= 0; --a)
    for (int b = o - a; b >= 0; --b) out.push_back(Exp3{a, b, o - a - b});
}

long multinomial(int a, int b, int c) {
  static const long fact[] = {1, 1, 2, 6, 24, 120, 720, 5040, 40320, 362880, 3628800, 39916800, 479001600};
  return fact[a + b + c] / (fact[a] * fact[b] * fact[c]);
}

struct Tensor {
  std::vector<int> open;  // open legs per canonical position
  int base;               // node id of component 0; components are contiguous, row-major
  int size;
};

struct Planner {
  std::map<std::pair<int, int>, int> basic_off;
  std::vector<std::array<int, 4>> prod;
  int n_nodes = 0;
  std::map<std::vector<int>, Tensor> memo;

  // per-graph state
  Adj a;
  std::vector<Label> labels;
  using VKey = std::array<int, 4>;
  struct Sub { bool done = false; std::vector<int> order, key; };
  Sub sub[128];
  long cost_[128];
  int split_[128];
  bool cost_done[128];

  int open_of(int v, unsigned mask) const {
    int o = labels[v][2];
    for (int w = 0; w < a.n; ++w) if (mask >> w & 1) o -= a.k[v][w];
    return o;
  }

  const Sub &canon(unsigned mask) {
    Sub &s = sub[mask];
    if (s.done) return s;
    std::vector<VKey> keys(a.n);
    std::vector<int> verts;
    for (int v = 0; v < a.n; ++v)
      if (mask >> v & 1) { keys[v] = VKey{labels[v][0], labels[v][1], labels[v][2], open_of(v, mask)}; verts.push_back(v); }
    std::sort(verts.begin(), verts.end(), [&](int x, int y) { return keys[x] < keys[y] || (keys[x] == keys[y] && x < y); });
    std::vector<int> ut;
    s.order = canonical_order<VKey>(a, verts, keys, &ut);
    s.key.clear();
    s.key.push_back((int)verts.size());
    for (int v : s.order) { s.key.push_back(keys[v][1]); s.key.push_back(keys[v][2]); s.key.push_back(keys[v][3]); }
    s.key.insert(s.key.end(), ut.begin(), ut.end());
    s.done = true;
    return s;
  }

  long merge_cost(unsigned s1, unsigned s2) {
    long c = 1;
    unsigned m = s1 | s2;
    for (int v = 0; v < a.n; ++v) if (m >> v & 1) c *= ncomp(open_of(v, m));
    for (int u = 0; u < a.n; ++u) if (s1 >> u & 1)
      for (int v = 0; v < a.n; ++v) if ((s2 >> v & 1) && a.k[u][v]) c *= ncomp(a.k[u][v]);
    return c;
  }

  long plan(unsigned mask) {
    if (cost_done[mask]) return cost_[mask];
    long best = -1; int bs = 0;
    if (__builtin_popcount(mask) == 1 || memo.count(canon(mask).key)) { best = 0; }
    else {
      unsigned low = mask & (~mask + 1);
      for (unsigned s1 = mask; s1; s1 = (s1 - 1) & mask) {
        if (!(s1 & low) || s1 == mask) continue;
        unsigned s2 = mask & ~s1;
        if (!connected(a, s1) || !connected(a, s2)) continue;
        long c = plan(s1) + plan(s2) + merge_cost(s1, s2);
        if (best < 0 || c < best) { best = c; bs = (int)s1; }
      }
    }
    cost_[mask] = best; split_[mask] = bs; cost_done[mask] = true;
    return best;
  }

  Tensor build(unsigned mask) {
    const Sub &s = canon(mask);
    if (__builtin_popcount(mask) == 1) {
      int v = s.order[0];
      Tensor t; t.open = {labels[v][2]}; t.base = basic_off.at({labels[v][1], labels[v][2]});
      t.size = ncomp(labels[v][2]);
      return t;
    }
    auto it = memo.find(s.key);
    if (it != memo.end()) return it->second;
    plan(mask);
    unsigned s1 = (unsigned)split_[mask], s2 = mask & ~s1;
    Tensor t1 = build(s1), t2 = build(s2);
    const std::vector<int> &o0 = canon(mask).order, &o1 = canon(s1).order, &o2 = canon(s2).order;
    Tensor t;
    t.size = 1;
    for (int v : o0) { int o = open_of(v, mask); t.open.push_back(o); t.size *= ncomp(o); }
    t.base = n_nodes;
    n_nodes += t.size;
    // bundles between s1 and s2
    struct Bundle { int u, v, k; };
    std::vector<Bundle> bundles;
    for (int u = 0; u < a.n; ++u) if (s1 >> u & 1)
      for (int v = 0; v < a.n; ++v) if ((s2 >> v & 1) && a.k[u][v]) bundles.push_back({u, v, a.k[u][v]});
    std::vector<std::vector<Exp3>> out_exps(o0.size()), bun_exps(bundles.size());
    for (size_t p = 0; p < o0.size(); ++p) list_exponents(t.open[p], out_exps[p]);
    for (size_t e = 0; e < bundles.size(); ++e) list_exponents(bundles[e].k, bun_exps[e]);
    std::vector<int> oi(o0.size(), 0);
    for (int comp = 0; comp < t.size; ++comp) {
      // decode comp -> per-position exponent choice (row-major, first position slowest)
      int rest = comp;
      for (int p = (int)o0.size() - 1; p >= 0; --p) { int d = (int)out_exps[p].size(); oi[p] = rest % d; rest /= d; }
      Exp3 ev[8];
      for (size_t p = 0; p < o0.size(); ++p) ev[o0[p]] = out_exps[p][oi[p]];
      std::vector<int> bi(bundles.size(), 0);
      while (true) {
        Exp3 tot[8];
        for (int v = 0; v < a.n; ++v) tot[v] = (mask >> v & 1) ? ev[v] : Exp3{0, 0, 0};
        long mult = 1;
        for (size_t e = 0; e < bundles.size(); ++e) {
          const Exp3 &x = bun_exps[e][bi[e]];
          mult *= multinomial(x.a, x.b, x.c);
          for (int w : {bundles[e].u, bundles[e].v}) { tot[w].a += x.a; tot[w].b += x.b; tot[w].c += x.c; }
        }
        auto index_in = [&](const Tensor &tt, const std::vector<int> &ord) {
          int idx = 0;
          for (size_t p = 0; p < ord.size(); ++p) {
            const Exp3 &x = tot[ord[p]];
            idx = idx * ncomp(tt.open[p]) + packed_index(x.a, x.b, x.c);
          }
          return tt.base + idx;
        };
        prod.push_back({index_in(t1, o1), index_in(t2, o2), (int)mult, t.base + comp});
        // next bundle assignment
        int e = (int)bundles.size() - 1;
        for (; e >= 0; --e) { if (++bi[e] < (int)bun_exps[e].size()) break; bi[e] = 0; }
        if (e < 0) break;
      }
    }
    memo[canon(mask).key] = t;
    return t;
  }

  int scalar(const Comp &c) {
    const int n = (int)c.labels.size();
    if (n == 1) return basic_off.at({c.labels[0][1], 0});
    a = to_matrix(n, c.ut);
    labels = c.labels;
    for (int m = 0; m < 128; ++m) { sub[m] = Sub(); cost_done[m] = false; }
    Tensor t = build((1u << n) - 1);
    return t.base;
  }
};

template <class T>
T *dup(const std::vector<T> &v) {
  T *p = (T *)std::malloc(sizeof(T) * (v.size() ? v.size() : 1));
  if (p && !v.empty()) std::memcpy(p, v.data(), sizeof(T) * v.size());
  return p;
}

}  // namespace

extern "C" int mtp_enumerate(int32_t lev_max, mtp_params *out) {
  if (!out || lev_max < 2 || lev_max > 28) return MTP_EINVAL;
  try {
    std::vector<Comp> comps = connected_scalars(lev_max);
    std::vector<Func> funcs = basis_functions(lev_max, comps);
    Planner pl;
    std::vector<int32_t> basic;
    int n_mu = 0;
    for (int mu = 0; 2 + 4 * mu <= lev_max; ++mu) {
      ++n_mu;
      for (int nu = 0;; ++nu) {
        bool ok = nu == 0 ? true : (4 * mu + 2 * nu <= lev_max - 4);
        if (!ok) break;
        pl.basic_off[{mu, nu}] = (int)basic.size() / 4;
        std::vector<Exp3> ex;
        list_exponents(nu, ex);
        for (auto &e : ex) { basic.push_back(mu); basic.push_back(e.a); basic.push_back(e.b); basic.push_back(e.c); }
      }
    }
    const int n_basic = (int)basic.size() / 4;
    pl.n_nodes = n_basic;
    std::vector<int> scalar_node(comps.size());
    for (size_t i = 0; i < comps.size(); ++i) scalar_node[i] = pl.scalar(comps[i]);
    std::map<std::vector<int>, int> func_node;
    std::vector<int32_t> basis_node, desc, desc_off;
    for (auto &f : funcs) {
      int node;
      if (f.comps.size() == 1) node = scalar_node[f.comps[0]];
      else {
        std::vector<int> prefix(f.comps.begin(), f.comps.end() - 1);
        node = pl.n_nodes++;
        pl.prod.push_back({func_node.at(prefix), scalar_node[f.comps.back()], 1, node});
      }
      func_node[f.comps] = node;
      basis_node.push_back(node);
      desc_off.push_back((int32_t)desc.size());
      desc.push_back((int32_t)f.comps.size());
      for (int ci : f.comps) {
        const Comp &c = comps[ci];
        desc.push_back((int32_t)c.labels.size());
        for (auto &l : c.labels) { desc.push_back(l[1]); desc.push_back(l[2]); }
        for (int k : c.ut) desc.push_back(k);
      }
    }
    desc_off.push_back((int32_t)desc.size());
    std::vector<int32_t> prod;
    for (auto &p : pl.prod) for (int x : p) prod.push_back(x);

    out->lev_max = lev_max;
    out->n_radial_funcs = n_mu;
    out->n_basic = n_basic;
    out->basic = dup(basic);
    out->n_nodes = pl.n_nodes;
    out->n_prod = (int32_t)pl.prod.size();
    out->prod = dup(prod);
    out->n_basis = (int32_t)funcs.size();
    out->basis_node = dup(basis_node);
    out->n_desc = (int32_t)desc.size();
    out->basis_desc = dup(desc);
    out->basis_desc_off = dup(desc_off);
    return MTP_OK;
  } catch (...) {
    return MTP_ENOMEM;
  }
}

extern "C" void mtp_table_free(mtp_params *t) {
  if (!t) return;
  std::free((void *)t->basic); std::free((void *)t->prod); std::free((void *)t->basis_node);
  std::free((void *)t->basis_desc); std::free((void *)t->basis_desc_off);
  t->basic = t->prod = t->basis_node = t->basis_desc = t->basis_desc_off = nullptr;
}
