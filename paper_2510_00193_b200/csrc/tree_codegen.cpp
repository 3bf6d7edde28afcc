// K2 code generation: contraction table -> straight-line register program for one atom per thread
// (tree_codegen.h explains the method).  BASELINE.json north_star: "a forward/adjoint contraction kernel with
// the tree in registers and shared memory"; the table is an input of mtp_create, so any valid table is accepted.
#include "tree_codegen.h"

#include <algorithm>
#include <cstdio>
#include <cstring>
#include <map>
#include <queue>

#include "mtp_b200.h"

namespace mtpb {

int k2_validate(int n_basic, int n_nodes, int n_prod, const int32_t *prod, int n_basis, const int32_t *basis_node,
                const char **err) {
  static const char *e_range = "contraction table: node index out of range";
  static const char *e_order = "contraction table: a node is read before its last write";
  static const char *e_mult = "contraction table: negative multiplicity";
  if (n_basic < 1 || n_nodes < n_basic || n_prod < 0 || (n_prod > 0 && !prod) || n_basis < 0 || (n_basis > 0 && !basis_node)) {
    *err = e_range; return MTP_EINVAL;
  }
  std::vector<int> last_write(n_nodes, -1), first_read(n_nodes, n_prod);
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
  return MTP_OK;
}

namespace {

// ---- virtual program: instructions over value ids (node values, adjoints, temporaries), no registers yet
struct VInst { int op, d, a, b, c, k, x; };   // op = K2Op (loads / stores of spills are added by the allocator)

struct Row {
  int dst = 0, pos = 0;
  std::vector<std::pair<int, std::vector<std::pair<int, int>>>> groups;   // (mult, terms), mult 1 first
};

struct Builder {
  const K2Table &t;
  const K2Kind kind;
  const int N, nb;
  const bool group;
  std::vector<VInst> v;
  std::vector<std::pair<int, int>> const_desc;
  std::map<uint64_t, int> cidx;
  int n_values;                            // VAL(n) = n, ADJ(n) = N + n, temporaries from 2N
  std::vector<Row> rows;
  std::vector<int> row_of;                 // node -> row index or -1
  std::vector<double> seed;                // constant seeds (whole / top): sum of xi over the functions on a node
  std::vector<char> seeded, is_cut, is_basis, needed, read_needed, adj_init;
  std::vector<int> cut_row_of, pending;
  bool any_energy = false;

  Builder(const K2Table &tt, K2Kind kk) : t(tt), kind(kk), N(tt.n_nodes), nb(tt.n_basic), group(tt.is_group()), n_values(2 * tt.n_nodes) {}
  int VAL(int n) const { return n; }
  int ADJ(int n) const { return N + n; }
  int temp() { return n_values++; }
  int in_row(int k) const { return t.in_row.empty() ? k : t.in_row[k]; }
  // constants are kept symbolically, mult * seed(node) (node = -1: the number mult itself), so that the program
  // text does not depend on the weights xi: one compiled kernel serves every potential with this table
  int konst(int node, int mult) {
    const uint64_t key = ((uint64_t)(uint32_t)(node + 1) << 32) | (uint32_t)mult;
    auto it = cidx.find(key);
    if (it != cidx.end()) return it->second;
    const_desc.push_back({node, mult});
    return cidx[key] = (int)const_desc.size() - 1;
  }
  void emit(int op, int d, int a = -1, int b = -1, int c = -1, int k = -1, int x = -1) { v.push_back(VInst{op, d, a, b, c, k, x}); }

  void build_rows() {
    const int np = t.n_prod();
    std::vector<int> last(N, -1);
    for (int i = 0; i < np; ++i) if (t.prod[4 * i + 2] > 0) last[t.prod[4 * i + 3]] = i;
    std::vector<int> order;
    for (int n = nb; n < N; ++n) if (last[n] >= 0) order.push_back(n);
    std::sort(order.begin(), order.end(), [&](int x, int y) { return last[x] < last[y]; });
    row_of.assign(N, -1);
    rows.resize(order.size());
    for (size_t r = 0; r < order.size(); ++r) { rows[r].dst = order[r]; rows[r].pos = last[order[r]]; row_of[order[r]] = (int)r; }
    for (int i = 0; i < np; ++i) {
      const int32_t *p = &t.prod[4 * i];
      if (p[2] <= 0) continue;
      Row &row = rows[row_of[p[3]]];
      size_t g = 0;
      while (g < row.groups.size() && row.groups[g].first != p[2]) ++g;
      if (g == row.groups.size()) row.groups.push_back({p[2], {}});
      row.groups[g].second.push_back({p[0], p[1]});
    }
    for (auto &row : rows)
      std::stable_sort(row.groups.begin(), row.groups.end(), [](const auto &x, const auto &y) { return x.first < y.first; });
  }

  void classify() {
    seed.assign(N, 0.0); seeded.assign(N, 0); is_cut.assign(N, 0); is_basis.assign(N, 0); cut_row_of.assign(N, -1);
    for (size_t a = 0; a < t.basis_node.size(); ++a) { seed[t.basis_node[a]] += t.xi[a]; is_basis[t.basis_node[a]] = 1; }
    for (int n = 0; n < N; ++n) seeded[n] = is_basis[n];              // whatever the value of its weight: see konst()
    for (size_t q = 0; q < t.cut_node.size(); ++q) { is_cut[t.cut_node[q]] = 1; cut_row_of[t.cut_node[q]] = t.cut_row[q]; }
    // a node is needed when it can reach an output: E_i (seeded), an exported basis value, or a cut node
    needed.assign(N, 0); read_needed.assign(N, 0);
    for (int n = 0; n < N; ++n)
      needed[n] = group ? is_cut[n] : (kind == K2_VALUES ? is_basis[n] : seeded[n]);
    for (int r = (int)rows.size() - 1; r >= 0; --r) {
      if (!needed[rows[r].dst]) continue;
      for (auto &g : rows[r].groups)
        for (auto &ab : g.second) { needed[ab.first] = needed[ab.second] = 1; read_needed[ab.first] = read_needed[ab.second] = 1; }
    }
    pending.assign(N, 0);
    for (auto &row : rows) {
      if (!needed[row.dst]) continue;
      for (auto &g : row.groups)
        for (auto &ab : g.second) { ++pending[ab.first]; ++pending[ab.second]; }
    }
    adj_init.assign(N, 0);
  }

  // the value of dst: sum over groups of mult * (sum of products); the group with multiplier 1 accumulates in place
  void forward_row(const Row &row) {
    const int d = row.dst;
    const bool energy_leaf = kind == K2_EF && !group && !read_needed[d];       // value only feeds E_i
    const bool want = read_needed[d] || (kind == K2_VALUES && (is_cut[d] || is_basis[d])) || (kind == K2_EF && !group && seeded[d]);
    if (!want) return;                    // e.g. the output scalars of a group in the adjoint pass: their value is not used
    bool have = false;                    // VAL(d) holds a partial sum
    for (auto &g : row.groups) {
      const int m = g.first;
      const bool direct = !energy_leaf && m == 1 && !have;
      const int acc = direct ? VAL(d) : temp();
      bool first = true;
      for (auto &ab : g.second) {
        if (first) emit(P_MUL, acc, VAL(ab.first), VAL(ab.second));
        else emit(P_FMA, acc, VAL(ab.first), VAL(ab.second), acc);
        first = false;
      }
      if (energy_leaf) { emit(P_ENERGY, -1, acc, -1, -1, konst(d, m)); any_energy = true; }
      else if (direct) have = true;
      else if (!have) { emit(P_MULK, VAL(d), acc, -1, -1, konst(-1, m)); have = true; }
      else if (m == 1) emit(P_ADD, VAL(d), acc, -1, VAL(d));
      else emit(P_FMAK, VAL(d), acc, -1, VAL(d), konst(-1, m));
    }
    if (energy_leaf) return;
    if (kind == K2_EF && !group && seeded[d]) { emit(P_ENERGY, -1, VAL(d), -1, -1, konst(d, 1)); any_energy = true; }
    if (kind == K2_VALUES) {
      if (group && is_cut[d]) emit(P_STS_OUT, -1, VAL(d), -1, -1, -1, cut_row_of[d]);
      if (!group && is_basis[d])
        for (size_t a = 0; a < t.basis_node.size(); ++a) if (t.basis_node[a] == d) emit(P_STB, -1, VAL(d), -1, -1, -1, (int)a);
    }
  }

  // ADJ(x) += s * VAL(other), s = a register value (sv >= 0) or the constant K[sk]
  void contribute(int x, int other, int sv, int sk, std::vector<int> &ready) {
    const int ax = ADJ(x);
    if (!adj_init[x]) {
      adj_init[x] = 1;
      bool have = true;
      if (x < nb && group) emit(P_LDOUT, ax, -1, -1, -1, -1, in_row(x));          // running sum over the groups
      else if (is_cut[x]) emit(P_LDSEED, ax, -1, -1, -1, -1, cut_row_of[x]);
      else if (!group && seeded[x]) emit(P_CONST, ax, -1, -1, -1, konst(x, 1));
      else have = false;
      if (!have) {
        if (sv >= 0) emit(P_MUL, ax, sv, VAL(other));
        else emit(P_MULK, ax, VAL(other), -1, -1, sk);
      } else {
        if (sv >= 0) emit(P_FMA, ax, sv, VAL(other), ax);
        else emit(P_FMAK, ax, VAL(other), -1, ax, sk);
      }
    } else {
      if (sv >= 0) emit(P_FMA, ax, sv, VAL(other), ax);
      else emit(P_FMAK, ax, VAL(other), -1, ax, sk);
    }
    if (--pending[x] == 0) {
      if (x < nb) emit(P_STOUT, -1, ax, -1, -1, -1, in_row(x));
      else ready.push_back(x);
    }
  }

  void backward_row(const Row &row, std::vector<int> &ready) {
    const int d = row.dst;
    const bool leaf = !read_needed[d] && !is_cut[d];            // adjoint = constant seed
    if (!leaf && !adj_init[d]) {                                  // a group's output scalar nothing below the cut reads
      emit(P_LDSEED, ADJ(d), -1, -1, -1, -1, cut_row_of[d]);
      adj_init[d] = 1;
    }
    for (auto &g : row.groups) {
      const int m = g.first;
      int sv = -1, sk = -1;
      if (leaf) sk = konst(d, m);
      else if (m == 1) sv = ADJ(d);
      else { sv = temp(); emit(P_MULK, sv, ADJ(d), -1, -1, konst(-1, m)); }
      for (auto &ab : g.second) {
        contribute(ab.first, ab.second, sv, sk, ready);
        contribute(ab.second, ab.first, sv, sk, ready);
      }
    }
  }

  void build() {
    build_rows();
    classify();
    // packed inputs that are outputs themselves
    for (int k = 0; k < nb; ++k) {
      if (kind == K2_EF && !group && seeded[k]) { emit(P_ENERGY, -1, VAL(k), -1, -1, konst(k, 1)); any_energy = true; }
      if (kind == K2_VALUES && !group && is_basis[k])
        for (size_t a = 0; a < t.basis_node.size(); ++a) if (t.basis_node[a] == k) emit(P_STB, -1, VAL(k), -1, -1, -1, (int)a);
    }
    std::vector<int> ready;
    for (auto &row : rows) {
      const int d = row.dst;
      if (!needed[d]) continue;
      forward_row(row);
      if (kind != K2_EF || pending[d] != 0) continue;
      ready.push_back(d);                  // adjoint of d is complete (a constant seed, or dE/dS of an output): eager sweep
      while (!ready.empty()) {
        const int x = ready.back();
        ready.pop_back();
        backward_row(rows[row_of[x]], ready);
      }
    }
    if (kind == K2_EF && !group)
      for (int k = 0; k < nb; ++k)
        if (!adj_init[k]) {                // a packed input no needed row reads: its adjoint is its own seed
          const int tv = temp();
          emit(P_CONST, tv, -1, -1, -1, (seeded[k] ? konst(k, 1) : konst(-1, 0)));
          emit(P_STOUT, -1, tv, -1, -1, -1, in_row(k));
        }
  }
};

// ---- register allocation: Belady replacement over the known trace
struct Allocator {
  const Builder &B;
  const int W, D;
  K2Gen &out;
  std::vector<std::vector<int>> uses;      // per value: instruction indices (ascending)
  std::vector<int> uptr;                   // first entry of uses[] not yet passed
  std::vector<int> reg_of, slot_of;
  std::vector<char> dirty, home_valid, loaded;
  std::vector<int> val_in_reg;
  std::priority_queue<int, std::vector<int>, std::greater<int>> free_slots;
  int n_slots = 0;
  static constexpr int INF = 1 << 30;

  Allocator(const Builder &b, int w, int d, K2Gen &o) : B(b), W(w), D(d), out(o) {}

  static void operands(const VInst &x, int *rd, int &nrd, int &wr) {
    nrd = 0; wr = -1;
    switch (x.op) {
      case P_LDIN: case P_LDSEED: case P_LDOUT: case P_CONST: wr = x.d; break;
      case P_STOUT: case P_STS_OUT: case P_STB: case P_ENERGY: rd[nrd++] = x.a; break;
      case P_MUL: rd[nrd++] = x.a; rd[nrd++] = x.b; wr = x.d; break;
      case P_FMA: rd[nrd++] = x.a; rd[nrd++] = x.b; rd[nrd++] = x.c; wr = x.d; break;
      case P_MULK: rd[nrd++] = x.a; wr = x.d; break;
      case P_FMAK: case P_ADD: rd[nrd++] = x.a; rd[nrd++] = x.c; wr = x.d; break;
      default: break;
    }
  }
  int next_use(int val, int i) {           // first use at an index > i
    const std::vector<int> &u = uses[val];
    int &p = uptr[val];
    while (p < (int)u.size() && u[p] <= i) ++p;
    return p < (int)u.size() ? u[p] : INF;
  }
  bool is_in(int val) const { return val < B.nb; }                              // VAL of a packed input
  bool is_out(int val) const { return val >= B.N && val < B.N + B.nb; }         // ADJ of a packed input
  void phys(int op, int d, int a, int b, int c, int k, int x) { out.prog.push_back(K2Inst{op, d, a, b, c, k, x}); }

  void release(int val) {
    const int r = reg_of[val];
    if (r >= 0) { val_in_reg[r] = -1; reg_of[val] = -1; }
  }
  void drop_slot(int val) {
    if (slot_of[val] >= 0) { free_slots.push(slot_of[val]); slot_of[val] = -1; }
    home_valid[val] = 0;
  }
  // a free register; pinned values (stamp == pin_stamp) are not evicted.  -1: none available
  int take_reg(int i, const std::vector<int> &pin, int pin_stamp) {
    for (int r = 0; r < W; ++r) if (val_in_reg[r] < 0) return r;
    int best = -1, best_nu = -1;
    for (int r = 0; r < W; ++r) {
      const int val = val_in_reg[r];
      if (pin[val] == pin_stamp) continue;
      const int nu = next_use(val, i - 1);        // uses at >= i count
      if (nu > best_nu) { best_nu = nu; best = r; }
    }
    if (best < 0) return -1;
    const int val = val_in_reg[best];
    if (best_nu < INF && dirty[val]) {
      if (is_out(val)) { phys(P_STOUT, -1, best, -1, -1, -1, B.in_row(val - B.N)); ++out.n_stg; }
      else {
        if (slot_of[val] < 0) {
          if (free_slots.empty()) free_slots.push(n_slots++);
          slot_of[val] = free_slots.top(); free_slots.pop();
        }
        phys(P_STS, -1, best, -1, -1, -1, slot_of[val]); ++out.n_sts;
      }
      home_valid[val] = 1; dirty[val] = 0;
    }
    val_in_reg[best] = -1; reg_of[val] = -1;
    return best;
  }
  // make an existing value resident (reload from its home); false: no register could be freed
  bool fetch(int val, int i, const std::vector<int> &pin, int pin_stamp) {
    if (reg_of[val] >= 0) return true;
    const int r = take_reg(i, pin, pin_stamp);
    if (r < 0) return false;
    if (is_in(val)) { phys(P_LDIN, r, -1, -1, -1, loaded[val] ? 1 : 0, B.in_row(val)); ++out.n_ldg; loaded[val] = 1; }
    else if (is_out(val)) { phys(P_LDOUT, r, -1, -1, -1, -1, B.in_row(val - B.N)); ++out.n_ldg; }
    else { phys(P_LDS, r, -1, -1, -1, -1, slot_of[val]); ++out.n_lds; }
    reg_of[val] = r; val_in_reg[r] = val; dirty[val] = 0;
    return true;
  }

  int run(std::string *err) {
    const std::vector<VInst> &v = B.v;
    const int n = (int)v.size(), nv = B.n_values;
    uses.assign(nv, {}); uptr.assign(nv, 0);
    reg_of.assign(nv, -1); slot_of.assign(nv, -1); dirty.assign(nv, 0); home_valid.assign(nv, 0); loaded.assign(nv, 0);
    val_in_reg.assign(W, -1);
    std::vector<char> exists(nv, 0);
    for (int k = 0; k < B.nb; ++k) { exists[k] = 1; home_valid[k] = 1; }          // packed inputs live in the input array
    int rd[3], nrd, wr;
    for (int i = 0; i < n; ++i) {
      operands(v[i], rd, nrd, wr);
      for (int q = 0; q < nrd; ++q) if (uses[rd[q]].empty() || uses[rd[q]].back() != i) uses[rd[q]].push_back(i);
      if (wr >= 0 && (uses[wr].empty() || uses[wr].back() != i)) uses[wr].push_back(i);
    }
    std::vector<int> pin(nv, -1);
    for (int i = 0; i < n; ++i) {
      // pin what the next D instructions read and is resident; this instruction's operands are loaded first
      operands(v[i], rd, nrd, wr);
      for (int q = 0; q < nrd; ++q) pin[rd[q]] = i;
      if (wr >= 0) pin[wr] = i;
      for (int q = 0; q < nrd; ++q) {
        if (!exists[rd[q]]) { *err = "k2 codegen: a value is read before it is defined"; return MTP_EINVAL; }
        if (!fetch(rd[q], i, pin, i)) { *err = "k2 codegen: register window too small"; return MTP_EUNSUP; }
      }
      for (int j = i + 1; j <= i + D && j < n; ++j) {          // reload ahead of use what is in a home right now
        int rd2[3], nrd2, wr2;
        operands(v[j], rd2, nrd2, wr2);
        for (int q = 0; q < nrd2; ++q) {
          const int val = rd2[q];
          if (reg_of[val] >= 0) { pin[val] = i; continue; }
          if (!exists[val] || !home_valid[val]) continue;
          if (fetch(val, i, pin, i)) pin[val] = i;
        }
      }
      // destination
      int rdst = -1;
      if (wr >= 0) {
        if (reg_of[wr] < 0) {
          const int r = take_reg(i, pin, i);
          if (r < 0) { *err = "k2 codegen: register window too small"; return MTP_EUNSUP; }
          reg_of[wr] = r; val_in_reg[r] = wr;
        }
        rdst = reg_of[wr];
        exists[wr] = 1; dirty[wr] = 1; home_valid[wr] = 0;
      }
      const VInst &x = v[i];
      auto R = [&](int val) { return val >= 0 ? reg_of[val] : -1; };
      switch (x.op) {
        case P_LDIN: ++out.n_ldg; dirty[wr] = 0; home_valid[wr] = 1; break;
        case P_LDSEED: ++out.n_ldg; break;
        case P_LDOUT: ++out.n_ldg; dirty[wr] = 0; home_valid[wr] = 1; break;
        case P_STOUT: case P_STS_OUT: case P_STB: ++out.n_stg; break;
        case P_CONST: break;
        default: ++out.n_arith; break;
      }
      phys(x.op, rdst, R(x.a), R(x.b), R(x.c), x.k, x.x);
      // values with no further use leave the window and give their slot back
      for (int q = 0; q <= nrd; ++q) {
        const int val = q < nrd ? rd[q] : wr;
        if (val < 0 || next_use(val, i) < INF) continue;
        release(val);
        if (!is_in(val)) drop_slot(val);
      }
    }
    out.n_regs = W; out.n_slots = n_slots;
    return MTP_OK;
  }
};

void emit_source(const Builder &B, K2Gen &g) {
  // multipliers and seeds: operands from the constant bank while it has room (8 KB, what its cache holds), else literals
  constexpr size_t kMaxConst = (size_t)kK2ConstBank;
  std::string &s = g.source;
  s.clear();
  s.reserve(g.prog.size() * 20 + 4096);
  char buf[160];
  auto K = [&](int k) {
    char t[48];
    // the multinomial multipliers 2, 3, 6, ... are immediate operands of DFMA / DMUL (their low word is zero); what
    // depends on the weights comes from the constant bank, filled when the kernel is loaded (K2Gen::consts), and
    // beyond its size from a table in global memory
    if (g.const_node[k] < 0) snprintf(t, sizeof t, "%d.0", g.const_mult[k]);
    else if ((size_t)k < kMaxConst) snprintf(t, sizeof t, "cm[%d]", k);
    else snprintf(t, sizeof t, "__ldg(a.cmx+%d)", k);
    return std::string(t);
  };
  snprintf(buf, sizeof buf, "__constant__ double cm[%zu];\n", std::min(kMaxConst, std::max<size_t>(g.const_node.size(), 1)));
  s += buf;
  snprintf(buf, sizeof buf, "#define K2_SLOTS %d\n#define K2_ENERGY %d\n", g.n_slots, g.writes_energy ? 1 : 0);
  s += buf;
  // what the CTA asks L2 for when it starts: the whole input block of its tile for a whole table or top program
  // (one bulk prefetch: config 4 tree time 0.68 -> 0.62 ms); nothing for a group program, which reads a subset of the
  // rows -- a prefetch per row was measured and costs more than it hides (level 24: tree 17.0 -> 19.0 ms)
  s += B.t.in_row.empty() ? "#define K2_PREFETCH PFALL();\n" : "#define K2_PREFETCH\n";
  std::string &b = g.body;
  b.clear();
  b.reserve(g.prog.size() * 20 + 4096);
  b += "  double ";
  for (int r = 0; r < g.n_regs; ++r) { snprintf(buf, sizeof buf, "r%d%s", r, r + 1 < g.n_regs ? "," : ";"); b += buf; if (r % 16 == 15) b += "\n  "; }
  b += "\n";
  for (const K2Inst &x : g.prog) {
    switch (x.op) {
      case P_LDIN: snprintf(buf, sizeof buf, x.k ? "  r%d=LR(%d);" : "  r%d=LI(%d);", x.d, x.x); break;
      case P_LDSEED: snprintf(buf, sizeof buf, "  r%d=LB(%d);", x.d, x.x); break;
      case P_LDOUT: snprintf(buf, sizeof buf, "  r%d=LO(%d);", x.d, x.x); break;
      case P_STOUT: snprintf(buf, sizeof buf, "  SO(%d,r%d);", x.x, x.a); break;
      case P_LDS: snprintf(buf, sizeof buf, "  r%d=LS(%d);", x.d, x.x); break;
      case P_STS: snprintf(buf, sizeof buf, "  SS(%d,r%d);", x.x, x.a); break;
      case P_MUL: snprintf(buf, sizeof buf, "  r%d=__dmul_rn(r%d,r%d);", x.d, x.a, x.b); break;
      case P_FMA: snprintf(buf, sizeof buf, "  r%d=fma(r%d,r%d,r%d);", x.d, x.a, x.b, x.c); break;
      case P_MULK: snprintf(buf, sizeof buf, "  r%d=__dmul_rn(%s,r%d);", x.d, K(x.k).c_str(), x.a); break;
      case P_FMAK: snprintf(buf, sizeof buf, "  r%d=fma(%s,r%d,r%d);", x.d, K(x.k).c_str(), x.a, x.c); break;
      case P_CONST: snprintf(buf, sizeof buf, "  r%d=%s;", x.d, K(x.k).c_str()); break;
      case P_ENERGY: snprintf(buf, sizeof buf, "  e=fma(%s,r%d,e);", K(x.k).c_str(), x.a); break;
      case P_STS_OUT: snprintf(buf, sizeof buf, "  SC(%d,r%d);", x.x, x.a); break;
      case P_STB: snprintf(buf, sizeof buf, "  SB(%d,r%d);", x.x, x.a); break;
      case P_ADD: snprintf(buf, sizeof buf, "  r%d=__dadd_rn(r%d,r%d);", x.d, x.a, x.c); break;
      default: buf[0] = 0; break;
    }
    b += buf;
    b += "\n";
  }
  (void)B;
}

}  // namespace

void k2_constants(const K2Table &t, K2Gen &g) {
  std::vector<double> seed(t.n_nodes, 0.0);
  for (size_t a = 0; a < t.basis_node.size(); ++a) seed[t.basis_node[a]] += t.xi[a];
  g.consts.resize(g.const_node.size());
  for (size_t k = 0; k < g.const_node.size(); ++k)
    g.consts[k] = g.const_node[k] < 0 ? (double)g.const_mult[k] : (double)g.const_mult[k] * seed[g.const_node[k]];
}

int k2_generate(const K2Table &t, K2Kind kind, int window, int lookahead, K2Gen &out, std::string *err) {
  out = K2Gen();
  const char *verr = "";
  int rc = k2_validate(t.n_basic, t.n_nodes, t.n_prod(), t.prod.data(), (int)t.basis_node.size(), t.basis_node.data(), &verr);
  if (rc != MTP_OK) { *err = verr; return rc; }
  if (t.basis_node.size() != t.xi.size() || t.cut_node.size() != t.cut_row.size() ||
      (!t.in_row.empty() && (int)t.in_row.size() != t.n_basic)) { *err = "k2 codegen: inconsistent table"; return MTP_EINVAL; }
  for (int c : t.cut_node) if (c < t.n_basic || c >= t.n_nodes) { *err = "k2 codegen: cut node out of range"; return MTP_EINVAL; }
  if (window < 8) { *err = "k2 codegen: register window too small"; return MTP_EINVAL; }
  Builder b(t, kind);
  b.build();
  out.writes_energy = b.any_energy || (kind == K2_EF && !t.is_group());
  Allocator a(b, window, lookahead, out);
  out.const_node.clear(); out.const_mult.clear();
  for (auto &cd : b.const_desc) { out.const_node.push_back(cd.first); out.const_mult.push_back(cd.second); }
  k2_constants(t, out);
  rc = a.run(err);
  if (rc != MTP_OK) return rc;
  emit_source(b, out);
  return MTP_OK;
}

}  // namespace mtpb
