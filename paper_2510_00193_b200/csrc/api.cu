// C ABI of the MTP hot path (include/mtp_b200.h): handle, table compilation, chunk scheduler
// (a10), variant selection and the launch sequences of
// mtp_compute / mtp_grade.  No CPU fallback: every numeric step runs in the CUDA kernels.
#include <cuda_runtime.h>

#include <new>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <map>
#include <memory>
#include <mutex>
#include <string>
#include <thread>
#include <tuple>
#include <vector>

#include "kernels.h"
#include "mtp_b200.h"
#include "stair.h"
#include "tree_partition.h"

using namespace mtpb;

namespace mtpb {
PairLevel pair_level_10();
PairLevel pair_level_16();
PairLevel pair_level_20();
PairLevel pair_level_24();
PairLevel pair_level_28();
const PairLevel *pair_level(int index) {
  static const PairLevel levels[] = {pair_level_10(), pair_level_16(), pair_level_20(), pair_level_24(),
                                     pair_level_28()};
  return (index >= 0 && index < kNumLevels) ? &levels[index] : nullptr;
}
}  // namespace mtpb

static thread_local std::string g_create_error;
void mtpb::set_thread_error(const char *msg) { g_create_error = msg ? msg : ""; }

struct mtp_handle {
  int S = 0, nb = 0, nmu = 0, n_basic = 0, n_nodes = 0, n_basis = 0, lev_max = 0;
  double r_min = 0, r_cut = 0;
  const PairLevel *pl = nullptr;
  int crow = 0;
  double *d_coef = nullptr, *d_xi = nullptr, *d_xi0 = nullptr;
  int *d_kmapF = nullptr, *d_kmapB = nullptr, *d_kmapS = nullptr, *d_basis_node = nullptr;
  int *d_flag = nullptr;                       // device counters: [0] rejected input pairs (MTP_INFO_INPUT_ERRORS), [1] pairs beyond the
                                               // per-pair scratch of a chunk (MTP_INFO_SCRATCH_OVERFLOW)
  int64_t chunk_pairs = 0;                     // MTP_OPT_CHUNK_PAIRS
  // K2 schedules, one per atom-lane count AL (compiled on first use; the large-N one at create)
  struct TreeDev {
    TreeSched sched;
    TreeTerm *d_fprog = nullptr, *d_bprog = nullptr;
    int *d_fwave = nullptr, *d_bwave = nullptr, *d_gseed_k = nullptr, *d_gzero_k = nullptr;
    int *d_eseed_slot = nullptr, *d_basis_slot = nullptr;
    double *d_adj_init = nullptr, *d_gseed_val = nullptr, *d_leaf_seed = nullptr, *d_eseed_val = nullptr;
    int *d_mload_k = nullptr, *d_cut_row = nullptr, *d_cut_vslot = nullptr, *d_cut_aslot = nullptr;
  };
  // A table the K2 kernels can run: the whole table, or -- when that leaves too few atoms per CTA -- the top
  // program and the group programs of its partition (tree_partition.cpp).  Host copies feed the compilations.
  struct Prog {
    int n_basic = 0, n_nodes = 0, n_basis = 0;
    std::vector<int32_t> prod, basis_node;
    std::vector<double> xi;
    std::vector<int32_t> basic_map, cut_local, cut_row;   // group programs only
    int slots[2][2] = {{0, 0}, {0, 0}};        // [elide][n_val, n_adj]
    std::map<int, TreeDev> trees;              // key: AL * 8 + AR * 2 + elide
    int n_prod() const { return (int)(prod.size() / 4); }
    bool is_group() const { return !cut_local.empty(); }
  };
  int codegen = 1;                             // MTP_OPT_TREE_CODEGEN
  // ---- K2, interpreter form (tree_kernel.cu): built on first use, i.e. only when the specialised kernels are
  // switched off or unavailable
  bool interp_ready = false;
  std::vector<Prog> progs;                     // [0] whole table; partitioned: [1] top, [2..] groups
  bool partitioned = false;
  // ---- K2, specialised form (tree_codegen.cpp + tree_jit.cpp): one register program per table, compiled at create
  struct JProg {
    K2Table table;
    K2Gen gen[2];                              // [K2_EF], [K2_VALUES]
    K2Kernel *kern[2] = {nullptr, nullptr};
  };
  std::vector<JProg> jprogs;                   // [0] whole table or top program; [1..] group programs
  bool jit_ready = false, jit_partitioned = false;
  std::string jit_note;                        // why the specialised kernels are not in use
  int n_jit_kernels = 0;
  // the table as given (host copy) and what both forms share of a partition
  K2Table whole;
  int n_cut_rows = 0;                          // rows of the cut-value arrays S / dE/dS
  int *d_gmap = nullptr;                       // [n_basic] cut row of a packed moment that is a cut node itself, else -1
  long long n_prod = 0;
  int64_t chunk_atoms = 0;
  int force_mode = MTP_FORCE_AUTO, variant = MTP_VARIANT_AUTO;
  std::string err;
  // staging for mtp_compute_host (grow-only), its copy / compute streams and chunk events
  void *stage = nullptr;
  size_t stage_bytes = 0;
  void *stage_nb = nullptr;                    // mtp_compute_host_pos: device list + its workspace (grow-only)
  size_t stage_nb_bytes = 0;
  int64_t nb_capacity = 0;                     // pairs the staged list holds
  cudaStream_t s_copy = nullptr, s_comp = nullptr;
  std::vector<cudaEvent_t> ev;
  std::vector<void *> to_free;
  // per-kernel-class device timing (MTP_OPT_PROFILE): event pairs recorded around each launch
  int profile = 0;
  int skin_list = 0;                            // MTP_OPT_SKIN_LIST: the caller's list carries pairs beyond R_cut
  struct Span { cudaEvent_t a, b; int cls; };
  std::vector<Span> spans;
  std::vector<cudaEvent_t> pool;
};

namespace {
enum { CLS_MOMENTS = 0, CLS_TREE = 1, CLS_PAIRGRAD = 2, CLS_OTHER = 3, CLS_GRADE = 4, N_CLS = 5 };
cudaEvent_t prof_event(mtp_handle *h) {
  if (!h->pool.empty()) { cudaEvent_t e = h->pool.back(); h->pool.pop_back(); return e; }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}
struct ProfScope {
  mtp_handle *h; cudaStream_t st; mtp_handle::Span s; bool on;
  ProfScope(mtp_handle *h_, int cls, cudaStream_t st_) : h(h_), st(st_), on(h_->profile != 0) {
    if (on) { s.a = prof_event(h); s.b = prof_event(h); s.cls = cls; cudaEventRecord(s.a, st); }
  }
  ~ProfScope() { if (on) { cudaEventRecord(s.b, st); h->spans.push_back(s); } }
};
}  // namespace
#define TIMED(h, cls, st, call) do { ProfScope ps__(h, cls, st); CU(h, call); } while (0)


static int fail(mtp_handle *h, int code, const std::string &msg) {
  if (h) h->err = msg; else g_create_error = msg;
  return code;
}
static int cuda_fail(mtp_handle *h, cudaError_t e, const char *where) {
  return fail(h, MTP_ECUDA, std::string(where) + ": " + cudaGetErrorString(e));
}
#define CU(h, call)                                                  \
  do {                                                               \
    cudaError_t e__ = (call);                                        \
    if (e__ != cudaSuccess) return cuda_fail(h, e__, #call);         \
  } while (0)

template <class T>
static cudaError_t upload(mtp_handle *h, T **dst, const T *src, size_t n) {
  cudaError_t e = cudaMalloc((void **)dst, sizeof(T) * std::max<size_t>(n, 1));
  if (e != cudaSuccess) return e;
  h->to_free.push_back(*dst);
  if (n) e = cudaMemcpy(*dst, src, sizeof(T) * n, cudaMemcpyHostToDevice);
  return e;
}

// ---- staircase helpers at run time (mirror stair.h) -----------------------------------
static int rt_numax(int lev, int mu) { int t = lev - 4 - 4 * mu; return t >= 2 ? t / 2 : 0; }
static int rt_nmu(int lev) { return (lev - 2) / 4 + 1; }
static bool rt_valid(int lev, int mu, int nu) { return mu < rt_nmu(lev) && (nu == 0 || rt_numax(lev, mu) >= nu); }
static int rt_nmu_for(int lev, int nu) {
  int n = 0;
  for (int mu = 0; mu < rt_nmu(lev); ++mu) if (nu == 0 || rt_numax(lev, mu) >= nu) ++n;
  return n;
}

// kmapF: slot order of k_moments (a, i, k, mu);  kmapB: slot order of k_pairgrad (mu, a desc, i desc, k desc)
static void build_kmaps(const PairLevel &pl, int n_basic, const int32_t *basic, std::vector<int> &kf,
                        std::vector<int> &kb) {
  const int lev = pl.lev, NSB = pl.nsb, NSC = pl.nsc, NS = NSB * NSC, NU0 = rt_numax(lev, 0);
  std::map<std::tuple<int, int, int, int>, int> where;
  for (int k = 0; k < n_basic; ++k) where[{basic[4 * k], basic[4 * k + 1], basic[4 * k + 2], basic[4 * k + 3]}] = k;
  auto find = [&](int mu, int a, int b, int c) {
    if (!rt_valid(lev, mu, a + b + c)) return -1;
    auto it = where.find({mu, a, b, c});
    return it == where.end() ? -1 : it->second;
  };
  kf.assign((size_t)NS * pl.nslot, -1);
  kb.assign((size_t)NS * pl.nslot, -1);
  for (int s = 0; s < NS; ++s) {
    const int sb = s % NSB, sc = s / NSB;
    int slot = 0;
    for (int a = 0; a <= NU0; ++a)
      for (int i = 0; i <= (NU0 - a) / NSB; ++i)
        for (int k = 0; k <= (NU0 - a - NSB * i) / NSC; ++k)
          for (int m = 0; m < rt_nmu_for(lev, a + NSB * i + NSC * k); ++m)
            kf[(size_t)s * pl.nslot + slot++] = find(m, a, sb + NSB * i, sc + NSC * k);
    slot = 0;
    for (int m = 0; m < rt_nmu(lev); ++m) {
      const int NUm = rt_numax(lev, m);
      for (int a = NUm; a >= 0; --a)
        for (int i = (NUm - a) / NSB; i >= 0; --i)
          for (int k = (NUm - a - NSB * i) / NSC; k >= 0; --k)
            kb[(size_t)s * pl.nslot + slot++] = find(m, a, sb + NSB * i, sc + NSC * k);
    }
  }
}

// K2 interpreter schedule of one program for a CTA shape (AL, AR) and leaf elision on/off: compiled from the host
// copy of its table and uploaded on first use
static int get_tree(mtp_handle *h, mtp_handle::Prog &pg, int AL, int AR, bool elide, const mtp_handle::TreeDev **out) {
  if (AL <= 0) return fail(h, MTP_EUNSUP, "contraction tree does not fit in shared memory");
  const int key = AL * 8 + AR * 2 + (elide ? 1 : 0);
  auto it = pg.trees.find(key);
  if (it != pg.trees.end()) { *out = &it->second; return MTP_OK; }
  mtp_handle::TreeDev td;
  const char *terr = "";
  const bool group = pg.is_group();
  int rc = tree_compile(pg.n_basic, pg.n_nodes, pg.n_prod(), pg.prod.data(), pg.n_basis, pg.basis_node.data(), pg.xi.data(),
                        AL * AR, tree_row_lanes(AL), elide, td.sched, &terr, group ? pg.basic_map.data() : nullptr,
                        group ? pg.cut_local.data() : nullptr, (int)pg.cut_local.size());
  if (rc != MTP_OK) return fail(h, rc, terr);
  cudaError_t e = cudaSuccess;
  auto up = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  const TreeSched &sc = td.sched;
  up(upload(h, &td.d_fprog, sc.fprog.data(), sc.fprog.size()));
  up(upload(h, &td.d_bprog, sc.bprog.data(), sc.bprog.size()));
  up(upload(h, &td.d_fwave, sc.fwave.data(), sc.fwave.size()));
  up(upload(h, &td.d_bwave, sc.bwave.data(), sc.bwave.size()));
  up(upload(h, &td.d_adj_init, sc.adj_init.data(), sc.adj_init.size()));
  up(upload(h, &td.d_leaf_seed, sc.leaf_seed.data(), sc.leaf_seed.size()));
  up(upload(h, &td.d_eseed_slot, sc.eseed_slot.data(), sc.eseed_slot.size()));
  up(upload(h, &td.d_eseed_val, sc.eseed_val.data(), sc.eseed_val.size()));
  up(upload(h, &td.d_basis_slot, sc.basis_slot.data(), sc.basis_slot.size()));
  up(upload(h, &td.d_gseed_k, sc.gseed_k.data(), sc.gseed_k.size()));
  up(upload(h, &td.d_gseed_val, sc.gseed_val.data(), sc.gseed_val.size()));
  up(upload(h, &td.d_gzero_k, sc.gzero_k.data(), sc.gzero_k.size()));
  if (group) {
    up(upload(h, &td.d_mload_k, sc.mload_k.data(), sc.mload_k.size()));
    up(upload(h, &td.d_cut_row, pg.cut_row.data(), pg.cut_row.size()));
    up(upload(h, &td.d_cut_vslot, sc.cut_val_slot.data(), sc.cut_val_slot.size()));
    up(upload(h, &td.d_cut_aslot, sc.cut_adj_slot.data(), sc.cut_adj_slot.size()));
  }
  if (e != cudaSuccess) return cuda_fail(h, e, "tree schedule upload");
  auto ins = pg.trees.emplace(key, std::move(td));
  *out = &ins.first->second;
  return MTP_OK;
}

extern "C" const char *mtp_last_error(const mtp_handle *h) { return h ? h->err.c_str() : g_create_error.c_str(); }
extern "C" int64_t mtp_launch_count(void) { return launch_count(); }

extern "C" int mtp_profile_read(mtp_handle *h, double *ms, int64_t *launches) {
  if (!h || !ms || !launches) return MTP_EINVAL;
  for (int c = 0; c < N_CLS; ++c) { ms[c] = 0.0; launches[c] = 0; }
  for (auto &s : h->spans) {
    if (cudaEventSynchronize(s.b) != cudaSuccess) return cuda_fail(h, cudaGetLastError(), "mtp_profile_read");
    float t = 0.f;
    cudaEventElapsedTime(&t, s.a, s.b);
    ms[s.cls] += t; launches[s.cls] += 1;
    h->pool.push_back(s.a); h->pool.push_back(s.b);
  }
  h->spans.clear();
  return MTP_OK;
}

extern "C" void mtp_destroy(mtp_handle *h) {
  if (!h) return;
  for (auto &s : h->spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
  for (auto e : h->pool) cudaEventDestroy(e);
  for (auto &jp : h->jprogs) for (auto *k : jp.kern) k2_jit_destroy(k);
  for (void *p : h->to_free) cudaFree(p);
  if (h->stage) cudaFree(h->stage);
  if (h->stage_nb) cudaFree(h->stage_nb);
  for (auto e : h->ev) cudaEventDestroy(e);
  if (h->s_copy) cudaStreamDestroy(h->s_copy);
  if (h->s_comp) cudaStreamDestroy(h->s_comp);
  delete h;
}

// ---- K2 set-up ------------------------------------------------------------------------------
// Interpreter form: a table whose monolithic evaluation gets fewer than 32 atoms per CTA is cut into a top program
// and group programs (tree_partition.cpp); budgets = shared-memory slots per atom that leave room for 64 (else 32)
// atoms per CTA beside the energy partials.
static bool interp_partition(const K2Table &t, TreePartition &part) {
  const int nb = (int)t.basis_node.size();
  bool ok = tree_partition(t.n_basic, t.n_nodes, t.n_prod(), t.prod.data(), nb, t.basis_node.data(), 430, part);
  if (!ok || part.groups.size() > 24)
    ok = tree_partition(t.n_basic, t.n_nodes, t.n_prod(), t.prod.data(), nb, t.basis_node.data(), 870, part);
  return ok;
}

static void prog_slots(mtp_handle::Prog &g) {
  for (int el = 0; el < 2; ++el)
    tree_count_slots(g.n_basic, g.n_nodes, g.n_prod(), g.prod.data(), el != 0, &g.slots[el][0], &g.slots[el][1],
                     g.cut_local.data(), (int)g.cut_local.size());
}

static int upload_gmap(mtp_handle *h, const TreePartition &part) {
  if (h->d_gmap) return MTP_OK;
  std::vector<int> gmap(h->n_basic, -1);
  for (size_t q = 0; q < part.cut_basic_k.size(); ++q) gmap[part.cut_basic_k[q]] = part.cut_basic_row[q];
  if (upload(h, &h->d_gmap, gmap.data(), gmap.size()) != cudaSuccess) return fail(h, MTP_ECUDA, "cut map upload");
  return MTP_OK;
}

static int ensure_interp(mtp_handle *h) {
  if (h->interp_ready) return MTP_OK;
  const K2Table &t = h->whole;
  h->progs.clear();
  h->progs.emplace_back();
  {
    mtp_handle::Prog &whole = h->progs.back();
    whole.n_basic = t.n_basic; whole.n_nodes = t.n_nodes; whole.n_basis = h->n_basis;
    whole.prod = t.prod; whole.basis_node = t.basis_node; whole.xi = t.xi;
    prog_slots(whole);
  }
  int AL = 0, AR = 1;
  tree_pick_shape(h->progs[0].slots[1][0], h->progs[0].slots[1][1], 0, &AL, &AR);
  TreePartition part;
  if (AL < 32 && interp_partition(t, part)) {
    h->partitioned = true;
    h->n_cut_rows = (int)part.cut_node.size();
    h->progs.emplace_back();
    {
      mtp_handle::Prog &top = h->progs.back();
      top.n_basic = part.top.n_basic; top.n_nodes = part.top.n_nodes; top.n_basis = h->n_basis;
      top.prod = part.top.prod; top.basis_node = part.top.basis_node; top.xi = t.xi;
      prog_slots(top);
    }
    for (auto &g : part.groups) {
      h->progs.emplace_back();
      mtp_handle::Prog &pg = h->progs.back();
      pg.n_basic = g.table.n_basic; pg.n_nodes = g.table.n_nodes; pg.n_basis = 0;
      pg.prod = g.table.prod; pg.basic_map = g.basic_map; pg.cut_local = g.cut_local; pg.cut_row = g.cut_row;
      prog_slots(pg);
    }
    int rc = upload_gmap(h, part);
    if (rc != MTP_OK) return rc;
  }
  for (size_t q = h->partitioned ? 1 : 0; q < h->progs.size(); ++q)
    for (int el = 0; el < 2; ++el) {
      tree_pick_shape(h->progs[q].slots[el][0], h->progs[q].slots[el][1], 0, &AL, &AR);
      if (AL == 0)
        return fail(h, MTP_EUNSUP, "contraction tree does not fit in shared memory (one atom's node values and adjoints > 225 KB)");
    }
  // build the large-system schedules now, so that errors surface here
  for (size_t q = h->partitioned ? 1 : 0; q < h->progs.size(); ++q) {
    const mtp_handle::TreeDev *td = nullptr;
    tree_pick_shape(h->progs[q].slots[1][0], h->progs[q].slots[1][1], 0, &AL, &AR);
    int rc = get_tree(h, h->progs[q], AL, AR, true, &td);
    if (rc != MTP_OK) return rc;
  }
  h->interp_ready = true;
  return MTP_OK;
}

// Specialised form.  A table whose register program needs more private shared memory than one 128-thread CTA per SM
// can have (kK2SlotsMax slots per thread) is cut below its product layer like for the interpreter; the group budget
// is chosen among a few by the estimated cost: arithmetic instructions of all programs, weighted by how few threads
// per SM their slot counts allow.
namespace {
struct JitPlan {
  bool partitioned = false;
  TreePartition part;
  std::vector<K2Table> tables;          // [0] whole or top, then groups
  double cost = 0.0;
  int min_threads = 0;                  // smallest threads-per-SM over the programs
};
double slots_penalty(int n_slots) {
  int threads = 0, ctas = 0;
  k2_shape(n_slots, &threads, &ctas);
  if (threads == 0) return 1e9;
  const int per_sm = threads * ctas;
  return per_sm >= 256 ? 1.0 : (per_sm >= 128 ? 1.5 : (per_sm >= 64 ? 3.0 : 6.0));
}
int threads_per_sm(int n_slots) { int t = 0, c = 0; k2_shape(n_slots, &t, &c); return t * c; }

K2Table group_table(const TreeGroup &g) {
  K2Table kt;
  kt.n_basic = g.table.n_basic; kt.n_nodes = g.table.n_nodes; kt.prod = g.table.prod; kt.in_row = g.basic_map;
  kt.cut_node = g.cut_local; kt.cut_row = g.cut_row;
  return kt;
}

// 0 or a negative code; err receives a message
int plan_jit(const K2Table &whole, JitPlan &best, std::string *err, bool *too_large = nullptr) {
  K2Gen g;
  int rc = k2_generate(whole, K2_EF, kK2Window, kK2Lookahead, g, err);
  if (rc != MTP_OK) return rc;
  best = JitPlan();
  if (g.n_slots <= kK2SlotsMax) {
    best.tables.push_back(whole);
    best.cost = (double)g.n_arith * slots_penalty(g.n_slots);
    best.min_threads = threads_per_sm(g.n_slots);
    return MTP_OK;
  }
  bool have = false;
  static const int budgets[] = {430, 600, 870};
  for (int budget : budgets) {
    JitPlan p;
    if (!tree_partition(whole.n_basic, whole.n_nodes, whole.n_prod(), whole.prod.data(), (int)whole.basis_node.size(),
                        whole.basis_node.data(), budget, p.part)) continue;
    p.partitioned = true;
    K2Table top;
    top.n_basic = p.part.top.n_basic; top.n_nodes = p.part.top.n_nodes; top.prod = p.part.top.prod;
    top.basis_node = p.part.top.basis_node; top.xi = whole.xi;
    p.tables.push_back(std::move(top));
    for (auto &gr : p.part.groups) p.tables.push_back(group_table(gr));
    bool ok = true;
    p.min_threads = 1 << 30;
    for (size_t q = 0; q < p.tables.size() && ok; ++q) {
      const int kinds = q == 0 ? 1 : 2;                 // groups run K2_VALUES and K2_EF in every evaluation
      for (int k = 0; k < kinds && ok; ++k) {
        K2Gen gq;
        std::string e2;
        if (k2_generate(p.tables[q], (K2Kind)k, kK2Window, kK2Lookahead, gq, &e2) != MTP_OK) { ok = false; break; }
        const double pen = slots_penalty(gq.n_slots);
        if (pen >= 1e9) { ok = false; break; }
        p.cost += (double)gq.n_arith * pen;
        p.min_threads = std::min(p.min_threads, threads_per_sm(gq.n_slots));
      }
    }
    if (!ok) continue;
    if (!have || p.cost < best.cost) { best = std::move(p); have = true; }
  }
  if (!have) { *err = "contraction table: no partition fits the specialised kernels"; return MTP_EUNSUP; }
  long long ops = 0;
  for (auto &t : best.tables) ops += t.n_prod();
  if (too_large) *too_large = ops > kK2MaxOps;
  if (ops > kK2MaxOps && !too_large) {   // level 28: 350 000 ops in 130 programs -- minutes of NVRTC time
    *err = "contraction table too large to specialise (" + std::to_string(ops) + " ops after partitioning): interpreted";
    return MTP_EUNSUP;
  }
  return MTP_OK;
}
}  // namespace

// Compiled kernels are kept for the life of the process, keyed by what the program text depends on (the table and
// its role, not the weights): a second potential with the same table costs no NVRTC time.
namespace {
struct CubinCache {
  std::mutex mu;
  std::map<std::pair<uint64_t, uint64_t>, std::shared_ptr<const std::vector<char>>> map;
};
CubinCache &cubin_cache() { static CubinCache c; return c; }
std::pair<uint64_t, uint64_t> program_key(const K2Table &t, int kind, int window, int lookahead) {
  uint64_t h1 = 1469598103934665603ull, h2 = 0x9e3779b97f4a7c15ull;
  auto mix = [&](int64_t v) {
    h1 = (h1 ^ (uint64_t)v) * 1099511628211ull;
    h2 = (h2 + (uint64_t)v) * 0xff51afd7ed558ccdull; h2 ^= h2 >> 33;
  };
  mix(kind); mix(window); mix(lookahead); mix(t.n_basic); mix(t.n_nodes);
  mix((int64_t)t.prod.size()); for (int32_t v : t.prod) mix(v);
  mix((int64_t)t.in_row.size()); for (int32_t v : t.in_row) mix(v);
  mix((int64_t)t.basis_node.size()); for (int32_t v : t.basis_node) mix(v);
  mix((int64_t)t.cut_node.size()); for (int32_t v : t.cut_node) mix(v);
  for (int32_t v : t.cut_row) mix(v);
  return {h1, h2};
}
}  // namespace

// Generates, compiles (in parallel: NVRTC takes about a second per thousand table ops) and loads the specialised kernels.
// On failure the handle stays usable through the interpreter; jit_note says why.
static int ensure_jit(mtp_handle *h) {
  if (h->jit_ready) return MTP_OK;
  std::string why;
  if (!k2_jit_available(&why)) { h->jit_note = why; return MTP_EUNSUP; }
  JitPlan plan;
  int rc = plan_jit(h->whole, plan, &why);
  if (rc != MTP_OK) { h->jit_note = why; return rc; }
  h->jprogs.clear();
  h->jprogs.resize(plan.tables.size());
  for (size_t q = 0; q < plan.tables.size(); ++q) h->jprogs[q].table = std::move(plan.tables[q]);
  h->jit_partitioned = plan.partitioned;
  if (plan.partitioned) {
    h->n_cut_rows = (int)plan.part.cut_node.size();
    rc = upload_gmap(h, plan.part);
    if (rc != MTP_OK) { h->jit_note = h->err; return rc; }
  }
  struct Job { mtp_handle::JProg *jp; int kind; std::shared_ptr<const std::vector<char>> cubin; std::string why; int rc = 0; };
  std::vector<Job> jobs;
  for (auto &jp : h->jprogs)
    for (int k = 0; k < 2; ++k) jobs.push_back(Job{&jp, k, nullptr, "", 0});
  std::atomic<size_t> next{0};
  const int window = kK2Window, lookahead = kK2Lookahead;
  auto work = [&]() {
    for (size_t i = next.fetch_add(1); i < jobs.size(); i = next.fetch_add(1)) {
      Job &j = jobs[i];
      j.rc = k2_generate(j.jp->table, (K2Kind)j.kind, window, lookahead, j.jp->gen[j.kind], &j.why);
      if (j.rc != MTP_OK) continue;
      const auto key = program_key(j.jp->table, j.kind, window, lookahead);
      {
        std::lock_guard<std::mutex> lk(cubin_cache().mu);
        auto it = cubin_cache().map.find(key);
        if (it != cubin_cache().map.end()) j.cubin = it->second;
      }
      if (!j.cubin) {
        auto bin = std::make_shared<std::vector<char>>(k2_jit_compile(j.jp->gen[j.kind], &j.why));
        if (bin->empty()) { j.rc = MTP_ECUDA; continue; }
        std::lock_guard<std::mutex> lk(cubin_cache().mu);
        cubin_cache().map[key] = bin;
        j.cubin = bin;
      }
      j.jp->gen[j.kind].body.clear(); j.jp->gen[j.kind].body.shrink_to_fit();      // the source is not needed any more
    }
  };
  std::vector<std::thread> workers;
  const unsigned hw = std::max(1u, std::thread::hardware_concurrency());
  for (unsigned t = 0; t < std::min<unsigned>(std::min(hw, 32u), (unsigned)jobs.size()); ++t) workers.emplace_back(work);
  for (auto &w : workers) w.join();
  for (auto &j : jobs) {
    if (j.rc == MTP_OK) {
      j.jp->kern[j.kind] = k2_jit_load(*j.cubin, j.jp->gen[j.kind].n_slots, j.jp->gen[j.kind].consts, &j.why);
      if (!j.jp->kern[j.kind]) j.rc = MTP_ECUDA;
    }
    if (j.rc != MTP_OK) {
      h->jit_note = j.why;
      for (auto &jp : h->jprogs) for (auto *&k : jp.kern) { k2_jit_destroy(k); k = nullptr; }
      h->jprogs.clear();
      return j.rc;
    }
  }
  h->n_jit_kernels = (int)jobs.size();
  h->jit_ready = true;
  return MTP_OK;
}

// Host-only diagnostic (no device needed): how mtp_create would evaluate this table with the specialised kernels.
extern "C" int mtp_table_plan(const mtp_params *p, int64_t *out) {
  if (!p || !out) return MTP_EINVAL;
  const char *verr = "";
  if (k2_validate(p->n_basic, p->n_nodes, p->n_prod, p->prod, p->n_basis, p->basis_node, &verr) != MTP_OK) return MTP_EINVAL;
  for (int q = 0; q < 8; ++q) out[q] = 0;
  K2Table whole;
  whole.n_basic = p->n_basic; whole.n_nodes = p->n_nodes; whole.prod.assign(p->prod, p->prod + 4 * (size_t)p->n_prod);
  whole.basis_node.assign(p->basis_node, p->basis_node + p->n_basis);
  whole.xi.assign((size_t)p->n_basis, 1.0);            // the plan does not depend on the weights (all taken non-zero)
  JitPlan plan;
  std::string err;
  bool too_large = false;
  int rc = plan_jit(whole, plan, &err, &too_large);
  if (rc != MTP_OK) return rc;
  out[0] = plan.partitioned ? 1 : 0;
  out[1] = plan.min_threads;
  out[7] = too_large ? 0 : 1;
  if (!plan.partitioned) return MTP_OK;
  out[2] = (int64_t)plan.part.cut_node.size(); out[3] = (int64_t)plan.part.groups.size(); out[4] = plan.part.top.n_prod();
  std::vector<char> seen(plan.part.cut_node.size(), 0);
  for (auto &g : plan.part.groups) {
    out[5] += g.table.n_prod();
    for (int r : g.cut_row) { if (r < 0 || r >= (int)seen.size() || seen[r]) return MTP_EINVAL; seen[r] = 1; }
  }
  for (size_t r = 0; r < seen.size(); ++r) if (!seen[r] && plan.part.cut_node[r] >= p->n_basic) return MTP_EINVAL;
  out[6] = (int64_t)p->n_prod - plan.part.top.n_prod();
  return MTP_OK;
}

extern "C" int mtp_create(mtp_handle **out, const mtp_params *p) {
  if (!out || !p) return fail(nullptr, MTP_EINVAL, "null argument");
  *out = nullptr;
  if (p->n_species < 1 || p->n_species > 16 || p->n_radial_basis < 1 || p->n_radial_basis > 16 ||
      p->n_radial_funcs < 1 || !(p->r_cut > p->r_min) || !(p->r_min >= 0) || p->n_basic < 1 ||
      p->n_nodes < p->n_basic || p->n_prod < 0 || p->n_basis < 1 || !p->basic || (p->n_prod && !p->prod) ||
      !p->basis_node || !p->c || !p->xi0 || !p->xi)
    return fail(nullptr, MTP_EINVAL, "mtp_params: bad sizes or null arrays");
  {                                   // the table is validated before anything walks it
    const char *verr = "";
    int rc = k2_validate(p->n_basic, p->n_nodes, p->n_prod, p->prod, p->n_basis, p->basis_node, &verr);
    if (rc != MTP_OK) return fail(nullptr, rc, verr);
  }
  int dev_count = 0;
  if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count == 0)
    return fail(nullptr, MTP_ECUDA, "no CUDA device: this library has no CPU fallback");
  // level of the pair kernels: the smallest compiled staircase containing every table tensor
  int li = -1;
  for (int c = 0; c < kNumLevels && li < 0; ++c) {
    bool ok = true;
    for (int k = 0; k < p->n_basic && ok; ++k) {
      const int32_t *b = p->basic + 4 * k;
      if (b[0] < 0 || b[1] < 0 || b[2] < 0 || b[3] < 0 || b[0] >= p->n_radial_funcs) return fail(nullptr, MTP_EINVAL, "basic: bad (mu,a,b,c)");
      ok = rt_valid(kLevels[c].lev, b[0], b[1] + b[2] + b[3]);
    }
    if (ok) li = c;
  }
  if (li < 0) return fail(nullptr, MTP_EUNSUP, "moment set exceeds the largest compiled level (28)");
  mtp_handle *h = new mtp_handle();
  h->S = p->n_species; h->nb = p->n_radial_basis; h->nmu = p->n_radial_funcs; h->n_basic = p->n_basic;
  h->n_nodes = p->n_nodes; h->n_basis = p->n_basis; h->lev_max = p->lev_max; h->r_min = p->r_min; h->r_cut = p->r_cut;
  h->pl = pair_level(li);
  h->n_prod = p->n_prod;
  h->whole.n_basic = p->n_basic; h->whole.n_nodes = p->n_nodes;
  h->whole.prod.assign(p->prod, p->prod + 4 * (size_t)p->n_prod);
  h->whole.basis_node.assign(p->basis_node, p->basis_node + p->n_basis);
  h->whole.xi.assign(p->xi, p->xi + p->n_basis);
  // radial coefficients: blocks (z_i, z_j) laid out [beta][NMUP], NMUP = the level's n_mu rounded up to even
  // (16-byte pairs); +2 doubles per block spread the blocks over the banks
  const int nmu_lev = rt_nmu(h->pl->lev), nmup = (nmu_lev + 1) & ~1;
  h->crow = nmup * h->nb + 2;
  // K1 / K3 stage the coefficients of every species pair in shared memory next to their pair tiles
  if ((size_t)h->S * h->S * h->crow * 8 + std::max(h->pl->smem_fixed, h->pl->smem_fixed_s) > 227 * 1024) {
    delete h;
    return fail(nullptr, MTP_EUNSUP, "n_species^2 x n_radial_basis x n_radial_funcs coefficients do not fit in shared memory beside the pair tiles");
  }
  std::vector<double> coef((size_t)h->S * h->S * h->crow, 0.0);
  for (int r = 0; r < h->S * h->S; ++r)
    for (int m = 0; m < h->nmu && m < nmu_lev; ++m)
      for (int b = 0; b < h->nb; ++b) coef[(size_t)r * h->crow + b * nmup + m] = p->c[((size_t)r * h->nmu + m) * h->nb + b];
  std::vector<int> kf, kb;
  build_kmaps(*h->pl, p->n_basic, p->basic, kf, kb);
  cudaError_t e = cudaSuccess;
  auto up = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  up(upload(h, &h->d_coef, coef.data(), coef.size()));
  up(upload(h, &h->d_xi, p->xi, (size_t)p->n_basis));
  up(upload(h, &h->d_xi0, p->xi0, (size_t)p->n_species));
  up(upload(h, &h->d_kmapF, kf.data(), kf.size()));
  up(upload(h, &h->d_kmapB, kb.data(), kb.size()));
  if (h->pl->nsl > 0) {                   // slot map of the sliced (large-system) pair kernels
    std::vector<int> ks((size_t)h->pl->nsl * h->pl->nslot_s, -1);
    h->pl->kmap_s(p->n_basic, p->basic, ks.data());
    up(upload(h, &h->d_kmapS, ks.data(), ks.size()));
  }
  up(upload(h, &h->d_basis_node, p->basis_node, (size_t)p->n_basis));
  {
    const int zero2[2] = {0, 0};
    up(upload(h, &h->d_flag, zero2, 2));
  }
  if (e != cudaSuccess) { int r = cuda_fail(nullptr, e, "mtp_create upload"); mtp_destroy(h); return r; }
  // K2: the specialised kernels; when they cannot be had (no NVRTC, ...) the reason is kept for mtp_last_error and
  // the interpreter is set up instead.  A table neither form can run fails here.
  int rc = ensure_jit(h);
  if (rc != MTP_OK) {
    rc = ensure_interp(h);
    if (rc != MTP_OK) { g_create_error = h->err; mtp_destroy(h); return rc; }
    h->err = "specialised contraction kernels not in use: " + h->jit_note;
  }
  *out = h;
  return MTP_OK;
}

extern "C" int mtp_set_option(mtp_handle *h, int key, int64_t v) {
  if (!h) return MTP_EINVAL;
  switch (key) {
    case MTP_OPT_CHUNK_ATOMS: if (v < 0) return fail(h, MTP_EINVAL, "chunk_atoms < 0"); h->chunk_atoms = v; return MTP_OK;
    case MTP_OPT_FORCE_MODE: if (v < 0 || v > 2) return fail(h, MTP_EINVAL, "bad force mode"); h->force_mode = (int)v; return MTP_OK;
    case MTP_OPT_VARIANT: if (v < 0 || v > 2) return fail(h, MTP_EINVAL, "bad variant"); h->variant = (int)v; return MTP_OK;
    case MTP_OPT_PROFILE: h->profile = v != 0; return MTP_OK;
    case MTP_OPT_SKIN_LIST: h->skin_list = v != 0; return MTP_OK;
    case MTP_OPT_CHUNK_PAIRS: if (v < 0) return fail(h, MTP_EINVAL, "chunk_pairs < 0"); h->chunk_pairs = v; return MTP_OK;
    case MTP_OPT_TREE_CODEGEN:
      if (v != 0 && !h->jit_ready) return fail(h, MTP_EUNSUP, "specialised contraction kernels not available: " + h->jit_note);
      if (v == 0) { int rc = ensure_interp(h); if (rc != MTP_OK) return rc; }
      h->codegen = v != 0; return MTP_OK;
  }
  return fail(h, MTP_EINVAL, "unknown option");
}
extern "C" int mtp_get_option(const mtp_handle *h, int key, int64_t *v) {
  if (!h || !v) return MTP_EINVAL;
  switch (key) {
    case MTP_OPT_CHUNK_ATOMS: *v = h->chunk_atoms; return MTP_OK;
    case MTP_OPT_FORCE_MODE: *v = h->force_mode; return MTP_OK;
    case MTP_OPT_VARIANT: *v = h->variant; return MTP_OK;
    case MTP_OPT_PROFILE: *v = h->profile; return MTP_OK;
    case MTP_OPT_SKIN_LIST: *v = h->skin_list; return MTP_OK;
    case MTP_OPT_TREE_CODEGEN: *v = h->codegen && h->jit_ready; return MTP_OK;
    case MTP_INFO_TREE_KERNELS: *v = h->jit_ready ? h->n_jit_kernels : 0; return MTP_OK;      // specialised K2 kernels loaded
    case MTP_INFO_TREE_PROGRAMS: *v = h->jit_ready ? (int64_t)h->jprogs.size() : 0; return MTP_OK;
    case MTP_OPT_CHUNK_PAIRS: *v = h->chunk_pairs; return MTP_OK;
    case MTP_INFO_INPUT_ERRORS:               // synchronises: pairs the packing kernel rejected since the last read
    case MTP_INFO_SCRATCH_OVERFLOW: {         // synchronises: pairs that did not fit a chunk's per-pair scratch
      const int q = key == MTP_INFO_INPUT_ERRORS ? 0 : 1;
      int flag = 0;
      if (cudaMemcpy(&flag, h->d_flag + q, sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess) return MTP_ECUDA;
      if (flag) cudaMemset(h->d_flag + q, 0, sizeof(int));
      *v = flag; return MTP_OK;
    }
  }
  return MTP_EINVAL;
}

// ---- chunk scheduler / workspace plan ---------------------------------------------------
namespace {
struct Plan {
  int64_t N = 0, nnz = 0, C = 0, cols = 0;      // cols: C rounded up to whole tiles of 128 atoms (kTile)
  int n_chunks = 0, P = 1, sliced = 0, atomic = 0, grid_chunk = 0, AL = 0, AR = 1, elide = 1;
  int64_t cap = 0;                              // pairs of one chunk the per-pair scratch (packed words, d4) holds
  size_t o_pos4 = 0, o_Ei = 0, o_M = 0, o_G = 0, o_wpart = 0, o_d4 = 0, o_B = 0, o_red = 0, o_idxp = 0, o_S = 0, o_Sbar = 0, o_jr = 0, o_korig = 0, o_cnt = 0, total = 0;
};
size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

// rows: atoms whose rows are evaluated (a window of the N atoms: mtp_compute_rows), -1 = all of them.  pos4 / Ei cover
// all N atoms, chunks and per-chunk scratch only the window.
int make_plan(const mtp_handle *h, int64_t n_all, int64_t nnz, int want_grade, int has_rev, Plan &pl, int64_t cap_exact = -1,
              int64_t rows = -1) {
  if (n_all < 0 || nnz < 0 || rows > n_all) return MTP_EINVAL;
  if (n_all > (1LL << 27)) return MTP_EUNSUP;      // neighbour words carry 27 index bits (pair_kernels.cuh)
  const int64_t N = rows < 0 ? n_all : rows;
  pl.N = N; pl.nnz = nnz;
  int64_t C = h->chunk_atoms;
  if (C <= 0) {
    // automatic: as few chunks as a budget of 4 GB for M + G (16 B x n_basic per atom) and 2^20 atoms allows -- every chunk
    // pays its own launches, tails and a walk of the rows it touches in the reverse gather (config 4, one B200: 4 / 2 /
    // 1 chunks -> 5.64 / 5.41 / 5.28 ms per step at 1.2 / 2.3 / 4.0 GB of workspace, 2 % of the 180 GB).  Callers
    // short of memory set MTP_OPT_CHUNK_ATOMS: 32 768 atoms -> 179 MB.
    C = std::min<int64_t>(1 << 20, (4LL << 30) / (16LL * h->n_basic));
    C = std::max<int64_t>(1024, C / 1024 * 1024);
    if (N > C) {  // equal chunks: no small last chunk
      const int64_t nc = (N + C - 1) / C;
      C = ((N + nc - 1) / nc + 31) / 32 * 32;
    }
  }
  if (C > N) C = std::max<int64_t>(N, 1);
  pl.C = C;
  pl.cols = (C + kTile - 1) / kTile * kTile;
  pl.n_chunks = N ? (int)((N + C - 1) / C) : 0;
  const int NS = h->pl->nsb * h->pl->nsc;
  if (h->variant == MTP_VARIANT_THREAD) pl.P = 1;
  else if (h->variant == MTP_VARIANT_BLOCK) pl.P = h->pl->p_small;
  else pl.P = (N * NS >= 2LL * 148 * 256) ? 1 : h->pl->p_small;   // fill the SMs' register files
  // PAPER.md:35 regimes: the thread-parallel mapping of a level that has the sliced kernels (pair_sliced.cuh: 32 atoms
  // per CTA, components across the warps) is those; the block-parallel one splits an atom's neighbours over lanes
  pl.sliced = pl.P == 1 && h->pl->nsl > 0 && h->d_kmapS != nullptr;
  pl.elide = want_grade ? 0 : 1;           // grades need every B_alpha stored
  if (h->interp_ready) tree_pick_shape(h->progs[0].slots[pl.elide][0], h->progs[0].slots[pl.elide][1], N, &pl.AL, &pl.AR);
  pl.atomic = h->force_mode == MTP_FORCE_ATOMIC || (h->force_mode == MTP_FORCE_AUTO && !has_rev);
  pl.grid_chunk = pl.sliced ? h->pl->pairgrad_grid_s((int)C) : h->pl->pairgrad_grid((int)C, pl.P);
  size_t o = 0;
  pl.o_pos4 = o; o = align_up(o + (size_t)n_all * 32);
  pl.o_Ei = o; o = align_up(o + (size_t)n_all * 8);
  pl.o_M = o; o = align_up(o + (size_t)h->n_basic * pl.cols * 8);
  pl.o_G = o; o = align_up(o + (size_t)h->n_basic * pl.cols * 8);
  pl.o_red = o; o = align_up(o + 2 * 256 * 8 * 8);            // partial rows of the two final sums (launch_reduce_energy_virial)
  if (h->n_cut_rows > 0) {                   // cut values and their adjoints of one chunk (tree_partition.cpp)
    pl.o_S = o; o = align_up(o + (size_t)h->n_cut_rows * pl.cols * 8);
    pl.o_Sbar = o; o = align_up(o + (size_t)h->n_cut_rows * pl.cols * 8);
  }
  // a10 (north_star "a chunk scheduler that bounds per-pair scratch"): packed neighbour words and d_ij
  // records exist for one chunk at a time.  The pair count of a chunk is known only on the device, so the buffers are
  // sized for MTP_OPT_CHUNK_PAIRS when set, else for 1.25 x the mean pairs per chunk + 4096 (lattice-like inputs; a
  // chunk that does not fit is counted in MTP_INFO_SCRATCH_OVERFLOW); a single chunk gets exactly nnz.
  if (pl.n_chunks <= 1) pl.cap = nnz;
  else if (cap_exact >= 0) pl.cap = cap_exact;
  else if (h->chunk_pairs > 0) pl.cap = std::min<int64_t>(nnz, h->chunk_pairs);
  else pl.cap = std::min<int64_t>(nnz, (int64_t)(1.25 * (double)nnz * (double)C / (double)std::max<int64_t>(N, 1)) + 4096);
  pl.o_idxp = o; o = align_up(o + (size_t)pl.cap * 4);        // packed neighbour words (used when shifts are given)
  pl.o_korig = o; o = align_up(o + (pl.sliced ? (size_t)pl.cap * 2 : 0));      // live rows (MTP_OPT_SKIN_LIST): CSR position of
  pl.o_cnt = o; o = align_up(o + (pl.sliced ? (size_t)pl.cols * 4 : 0));       // a compacted entry, live entries per atom
  pl.o_jr = o; o = align_up(o + kTouchWords * sizeof(unsigned));      // touch bitmap of the current chunk
  pl.o_wpart = o; o = align_up(o + (size_t)std::max(1, pl.n_chunks) * pl.grid_chunk * 64);
  pl.o_d4 = o; if (!want_grade && !pl.atomic) o = align_up(o + (size_t)pl.cap * 32);
  pl.o_B = o; if (want_grade) o = align_up(o + (size_t)pl.cols * h->n_basis * 8);      // tiled Bt of one chunk
  pl.total = o;
  return MTP_OK;
}

int box_setup(mtp_handle *h, const double *box, bool need_minimg, double r_cut, PairArgs &pa) {
  const double *a = box, *b = box + 3, *c = box + 6;
  const double bc[3] = {b[1] * c[2] - b[2] * c[1], b[2] * c[0] - b[0] * c[2], b[0] * c[1] - b[1] * c[0]};
  const double ca[3] = {c[1] * a[2] - c[2] * a[1], c[2] * a[0] - c[0] * a[2], c[0] * a[1] - c[1] * a[0]};
  const double ab[3] = {a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]};
  const double vol = a[0] * bc[0] + a[1] * bc[1] + a[2] * bc[2];
  for (int i = 0; i < 9; ++i) pa.H[i] = box[i];
  if (!(std::fabs(vol) > 0)) {
    if (need_minimg) return fail(h, MTP_EBOX, "singular box");
    for (int i = 0; i < 9; ++i) pa.Hi[i] = 0;
    return MTP_OK;
  }
  // H^-1 (row-vector convention: frac = cart . Hi): columns are bc, ca, ab over vol
  for (int i = 0; i < 3; ++i) { pa.Hi[3 * i + 0] = bc[i] / vol; pa.Hi[3 * i + 1] = ca[i] / vol; pa.Hi[3 * i + 2] = ab[i] / vol; }
  if (need_minimg) {
    auto norm = [](const double *v) { return std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]); };
    const double hmin = std::min({std::fabs(vol) / norm(bc), std::fabs(vol) / norm(ca), std::fabs(vol) / norm(ab)});
    if (!(hmin > 2.0 * r_cut)) return fail(h, MTP_EBOX, "box height < 2 R_cut and no image shifts given");
  }
  return MTP_OK;
}

// idx: the packed neighbour words when shifts were given (launch_pack_pairs), else the caller's plain indices
void fill_pair_args(const mtp_handle *h, PairArgs &pa, const double *pos4, const int64_t *off, const int32_t *idx,
                    const int8_t *shift) {
  pa.pos4 = pos4; pa.off = (const long long *)off; pa.idx = idx;
  pa.coef = h->d_coef; pa.n_species = h->S; pa.nb = h->nb; pa.crow = h->crow;
  pa.minimg = shift ? 0 : 1; pa.r_min = h->r_min; pa.r_cut = h->r_cut; pa.inv_width = 1.0 / (h->r_cut - h->r_min);
  pa.M = nullptr; pa.G = nullptr; pa.d4 = nullptr; pa.F = nullptr; pa.wpart = nullptr; pa.kmap = nullptr;
  pa.d4_cap = 0; pa.flag = h->d_flag; pa.idx_rel = 0; pa.idx_cap = 1LL << 62; pa.cnt = nullptr; pa.korig = nullptr;
}

// One chunk of K2 work: B_alpha / E_i (forward) and, when want_adj, G = dE_i/dM.  B != null: every basis value of
// the chunk is exported as the tiled Bt (no leaf elision).  All arrays are chunk-relative and tiled (kTile).
struct K2Io {
  const double *pos4; const double *M; double *G; double *Ei; double *B;
  int c0, c1; int want_adj; int64_t N; double *S; double *Sbar;
};

// interpreter: one launch of program pg
int launch_prog(mtp_handle *h, mtp_handle::Prog &pg, const K2Io &io, bool elide, const double *M, double *G, int n_rows,
                int want_adj, double *S, const double *Sbar, int g_accum, int write_energy, double *B, cudaStream_t st) {
  int AL = 0, AR = 1;
  tree_pick_shape(pg.slots[elide][0], pg.slots[elide][1], io.N, &AL, &AR);
  const mtp_handle::TreeDev *td = nullptr;
  int rc = get_tree(h, pg, AL, AR, elide, &td);
  if (rc != MTP_OK) return rc;
  const TreeSched &sc = td->sched;
  TreeArgs ta;
  ta.fprog = td->d_fprog; ta.fwave = td->d_fwave; ta.nfw = (int)sc.fwave.size() - 1;
  ta.bprog = td->d_bprog; ta.bwave = td->d_bwave; ta.nbw = (int)sc.bwave.size() - 1;
  ta.n_fprog = (int)sc.fprog.size(); ta.n_bprog = (int)sc.bprog.size(); ta.prog_smem_off = 0;
  ta.xi0 = h->d_xi0; ta.pos4 = io.pos4;
  ta.adj_init = td->d_adj_init; ta.leaf_seed = td->d_leaf_seed;
  ta.eseed_slot = td->d_eseed_slot; ta.eseed_val = td->d_eseed_val; ta.n_eseed = (int)sc.eseed_slot.size();
  ta.basis_slot = td->d_basis_slot;
  ta.gseed_k = td->d_gseed_k; ta.gseed_val = td->d_gseed_val; ta.n_gseed = (int)sc.gseed_k.size();
  ta.gzero_k = td->d_gzero_k; ta.n_gzero = (int)sc.gzero_k.size();
  ta.n_val = sc.n_val; ta.n_adj = sc.n_adj; ta.n_basic = pg.n_basic; ta.n_basis = pg.n_basis;
  ta.M = M; ta.G = G; ta.n_rows = n_rows; ta.n_cut_rows = h->n_cut_rows;
  ta.Ei = io.Ei; ta.B = B; ta.c0 = io.c0; ta.c1 = io.c1; ta.want_adj = want_adj;
  ta.mload_k = td->d_mload_k; ta.cut_row = td->d_cut_row; ta.cut_vslot = td->d_cut_vslot; ta.cut_aslot = td->d_cut_aslot;
  ta.n_cut = (int)pg.cut_local.size();
  ta.S = S; ta.Sbar = Sbar; ta.g_accum = g_accum; ta.write_energy = write_energy;
  TIMED(h, CLS_TREE, st, launch_tree(ta, AL, AR, st));
  return MTP_OK;
}

// A partitioned table runs its group programs forward, the top program, and the group programs again forward +
// backward seeded with the top program's adjoints (tree_partition.cpp).
int run_k2_interp(mtp_handle *h, const K2Io &io, cudaStream_t st) {
  int rc = ensure_interp(h);
  if (rc != MTP_OK) return rc;
  const bool elide = io.B == nullptr;
  if (!h->partitioned)
    return launch_prog(h, h->progs[0], io, elide, io.M, io.G, h->n_basic, io.want_adj, nullptr, nullptr, 0, 1, io.B, st);
  CU(h, launch_scopy(io.S, h->n_cut_rows, h->n_basic, io.c1 - io.c0, h->d_gmap, io.M, st));
  for (size_t q = 2; q < h->progs.size() && rc == MTP_OK; ++q)
    rc = launch_prog(h, h->progs[q], io, true, io.M, nullptr, h->n_basic, 0, io.S, nullptr, 0, 0, nullptr, st);
  if (rc != MTP_OK) return rc;
  rc = launch_prog(h, h->progs[1], io, elide, io.S, io.Sbar, h->n_cut_rows, io.want_adj, nullptr, nullptr, 0, 1, io.B, st);
  if (rc != MTP_OK || !io.want_adj) return rc;
  CU(h, launch_ginit(io.G, h->n_cut_rows, h->n_basic, io.c1 - io.c0, h->d_gmap, io.Sbar, st));
  for (size_t q = 2; q < h->progs.size() && rc == MTP_OK; ++q)
    rc = launch_prog(h, h->progs[q], io, true, io.M, io.G, h->n_basic, 1, nullptr, io.Sbar, 1, 0, nullptr, st);
  return rc;
}

// specialised kernels: K2_VALUES exports (B or the cut values), K2_EF does energy + adjoint
int run_k2_jit(mtp_handle *h, const K2Io &io, cudaStream_t st) {
  K2Args ka;
  ka.in = io.M; ka.out = io.G; ka.sbar = nullptr; ka.sout = nullptr; ka.bt = io.B; ka.Ei = io.Ei;
  ka.xi0 = h->d_xi0; ka.pos4 = io.pos4;
  ka.n_io = h->n_basic; ka.n_cut = h->n_cut_rows; ka.n_bt = h->n_basis; ka.c0 = io.c0; ka.n = io.c1 - io.c0;
  const bool want_ef = io.want_adj || !io.B;
  if (!h->jit_partitioned) {
    if (io.B) TIMED(h, CLS_TREE, st, k2_jit_launch(h->jprogs[0].kern[K2_VALUES], ka, st));
    if (want_ef) TIMED(h, CLS_TREE, st, k2_jit_launch(h->jprogs[0].kern[K2_EF], ka, st));
    return MTP_OK;
  }
  CU(h, launch_scopy(io.S, h->n_cut_rows, h->n_basic, io.c1 - io.c0, h->d_gmap, io.M, st));
  ka.sout = io.S;
  for (size_t q = 1; q < h->jprogs.size(); ++q) TIMED(h, CLS_TREE, st, k2_jit_launch(h->jprogs[q].kern[K2_VALUES], ka, st));
  K2Args kt = ka;                              // top program: inputs = cut values, adjoints = dE/dS
  kt.in = io.S; kt.out = io.Sbar; kt.n_io = h->n_cut_rows; kt.sout = nullptr;
  if (io.B) TIMED(h, CLS_TREE, st, k2_jit_launch(h->jprogs[0].kern[K2_VALUES], kt, st));
  if (want_ef) TIMED(h, CLS_TREE, st, k2_jit_launch(h->jprogs[0].kern[K2_EF], kt, st));
  if (!io.want_adj) return MTP_OK;
  CU(h, launch_ginit(io.G, h->n_cut_rows, h->n_basic, io.c1 - io.c0, h->d_gmap, io.Sbar, st));
  ka.sout = nullptr; ka.sbar = io.Sbar;
  for (size_t q = 1; q < h->jprogs.size(); ++q) TIMED(h, CLS_TREE, st, k2_jit_launch(h->jprogs[q].kern[K2_EF], ka, st));
  return MTP_OK;
}

int run_k2(mtp_handle *h, const K2Io &io, cudaStream_t st) {
  return (h->codegen && h->jit_ready) ? run_k2_jit(h, io, st) : run_k2_interp(h, io, st);
}
}  // namespace

extern "C" int mtp_workspace_bytes(const mtp_handle *h, int64_t n_atoms, int64_t nnz, int want_grade, size_t *out) {
  if (!h || !out) return MTP_EINVAL;
  Plan pl;
  int rc = make_plan(h, n_atoms, nnz, want_grade, /*has_rev=*/1, pl);
  if (rc != MTP_OK) return rc;
  *out = pl.total + 256 + (want_grade ? align_up((size_t)h->n_basis * 8) : 0);
  return MTP_OK;
}

// Pipelining hooks of mtp_compute_host: the pairs of chunk c (device arrays idx / shift, filled by an asynchronous
// copy on another stream) are ready when chunk_ready[c] has fired, rev when rev_ready has; chunk_pair0[c] is the
// CSR offset of the chunk's first atom (host copy), so that the neighbour words are packed chunk by chunk.
struct HostPipe {
  const std::vector<cudaEvent_t> *chunk_ready = nullptr;
  const std::vector<long long> *chunk_pair0 = nullptr;    // n_chunks + 1 entries
  cudaEvent_t rev_ready = nullptr;
};

static int compute_impl(mtp_handle *h, int64_t N, const double *d_pos, const int32_t *d_type, const double *box,
                        const int64_t *d_off, const int32_t *d_idx, const int8_t *d_shift, const int32_t *d_rev,
                        int64_t nnz, double *d_E, double *d_Ei, double *d_F, double *d_virial, void *d_ws,
                        size_t ws_bytes, void *stream, const HostPipe *pipe, int64_t cap_exact = -1, int64_t row_lo = 0,
                        int64_t row_hi = -1) {
  // [row_lo, row_hi): the atoms whose rows this call evaluates (mtp_compute_rows; d_off then is the window's own CSR,
  // d_off[0] = 0); the default is all of them
  if (!h) return MTP_EINVAL;
  if (!box || !d_E || (N > 0 && (!d_pos || !d_type || !d_off || !d_F)) || (nnz > 0 && !d_idx))
    return fail(h, MTP_EINVAL, "mtp_compute: null argument");
  if (h->force_mode == MTP_FORCE_GATHER && !d_rev && nnz > 0) return fail(h, MTP_EINVAL, "gather mode needs d_rev");
  cudaStream_t st = (cudaStream_t)stream;
  const bool window = row_hi >= 0;
  if (!window) { row_lo = 0; row_hi = N; }
  if (row_lo < 0 || row_hi < row_lo || row_hi > N) return fail(h, MTP_EINVAL, "row window outside [0, n_atoms]");
  d_off -= row_lo;                               // the kernels index offsets by atom
  Plan pl;
  int rc = make_plan(h, N, nnz, 0, d_rev != nullptr, pl, cap_exact, window ? row_hi - row_lo : -1);
  if (rc != MTP_OK) return fail(h, rc, "bad sizes");
  if (window && !pl.atomic) return fail(h, MTP_EINVAL, "a row window has no reverse pairs to gather: MTP_FORCE_ATOMIC or MTP_FORCE_AUTO");
  const size_t base = align_up((size_t)(uintptr_t)d_ws) - (size_t)(uintptr_t)d_ws;
  if (N > 0 && (!d_ws || ws_bytes < pl.total + base)) return fail(h, MTP_ESIZE, "workspace too small");
  PairArgs pa;
  rc = box_setup(h, box, d_shift == nullptr && nnz > 0, h->r_cut, pa);
  if (rc != MTP_OK) return rc;
  if (N == 0) {
    CU(h, launch_zero(d_E, 1, st));
    if (d_virial) CU(h, launch_zero(d_virial, 6, st));
    return MTP_OK;
  }
  char *ws = (char *)d_ws + base;
  double *pos4 = (double *)(ws + pl.o_pos4), *Ei = d_Ei ? d_Ei : (double *)(ws + pl.o_Ei);
  double *M = (double *)(ws + pl.o_M), *G = (double *)(ws + pl.o_G), *wpart = (double *)(ws + pl.o_wpart);
  double *d4 = (double *)(ws + pl.o_d4);
  int *idxp = (int *)(ws + pl.o_idxp);
  unsigned *jrange = (unsigned *)(ws + pl.o_jr);
  // pos4, F = 0 (both force modes accumulate: atomics, or chunk by chunk in fixed order), virial partials = 0, the first
  // chunk's touch bitmap = 0: one launch
  CU(h, launch_prologue(d_pos, d_type, (int)N, pos4, d_F, wpart, (long long)pl.n_chunks * pl.grid_chunk * 8, jrange, st));
  // MTP_OPT_SKIN_LIST (large-system kernels only): rows compacted to the entries within R_cut, chunk by chunk
  const bool live = h->skin_list && pl.sliced && nnz > 0;
  unsigned short *korig = (unsigned short *)(ws + pl.o_korig);
  int *cnt = (int *)(ws + pl.o_cnt);
  fill_pair_args(h, pa, pos4, d_off, (d_shift || live) ? idxp : d_idx, d_shift);
  pa.n_rows = h->n_basic;
  pa.idx_rel = (d_shift || live) ? 1 : 0;        // packed words exist for the current chunk only
  pa.idx_cap = (d_shift || live) ? pl.cap : nnz;
  pa.d4_cap = pl.cap;
  K2Io io{pos4, M, G, Ei, nullptr, 0, 0, 1, N, (double *)(ws + pl.o_S), (double *)(ws + pl.o_Sbar)};
  bool rev_waited = false;
  for (int c = 0; c < pl.n_chunks; ++c) {
    pa.c0 = (int)(row_lo + c * pl.C); pa.c1 = (int)std::min<int64_t>(row_hi, row_lo + (c + 1) * pl.C);
    if (pipe) CU(h, cudaStreamWaitEvent(st, (*pipe->chunk_ready)[c], 0));      // this chunk's pairs have arrived
    // the chunk's neighbour words (validated, index + image code in 4 bytes) and the range of atoms it touches
    if (live)
      CU(h, launch_pack_rows_live(pa, d_idx, (const signed char *)d_shift, N, pl.cap, idxp, korig, cnt, pl.atomic ? nullptr : d4, jrange, st,
                                  c == 0));
    else if (nnz > 0)
      CU(h, launch_pack_pairs_chunk((const long long *)d_off, pa.c0, pa.c1, d_idx, (const signed char *)d_shift, N, pl.cap,
                                    d_shift ? idxp : nullptr, h->d_flag, jrange, st, c == 0));
    pa.cnt = live ? cnt : nullptr; pa.korig = live ? korig : nullptr;
    pa.M = M; pa.G = G; pa.kmap = pl.sliced ? h->d_kmapS : h->d_kmapF;
    TIMED(h, CLS_MOMENTS, st, (pl.sliced ? h->pl->moments_s(pa, st) : h->pl->moments(pa, pl.P, st)));
    io.c0 = pa.c0; io.c1 = pa.c1;
    rc = run_k2(h, io, st);
    if (rc != MTP_OK) return rc;
    pa.kmap = pl.sliced ? h->d_kmapS : h->d_kmapB; pa.wpart = wpart + (size_t)c * pl.grid_chunk * 8;
    pa.d4 = pl.atomic ? nullptr : d4; pa.F = d_F;
    TIMED(h, CLS_PAIRGRAD, st, (pl.sliced ? h->pl->pairgrad_s(pa, pl.atomic, st) : h->pl->pairgrad(pa, pl.P, pl.atomic, st, nullptr)));
    if (!pl.atomic && nnz > 0) {                 // a8: this chunk's share of every F_k it touches, chunks in stream order
      if (pipe && pipe->rev_ready && !rev_waited) { CU(h, cudaStreamWaitEvent(st, pipe->rev_ready, 0)); rev_waited = true; }
      TIMED(h, CLS_OTHER, st, launch_gather_chunk((const long long *)d_off, d_idx, d_rev, d4, pl.cap, pa.c0, pa.c1, (int)N, jrange, d_F, st));
    }
  }
  double *red = (double *)(ws + pl.o_red);
  // E = sum of the window's E_i (an empty window sums nothing: 0) and the virial from the block partials, in one launch
  CU(h, launch_reduce_energy_virial(Ei + row_lo, row_hi - row_lo, d_E, wpart, (long long)pl.n_chunks * pl.grid_chunk, d_virial, red, st));
  return MTP_OK;
}

extern "C" int mtp_compute(mtp_handle *h, int64_t N, const double *d_pos, const int32_t *d_type, const double *box,
                           const int64_t *d_off, const int32_t *d_idx, const int8_t *d_shift, const int32_t *d_rev,
                           int64_t nnz, double *d_E, double *d_Ei, double *d_F, double *d_virial, void *d_ws,
                           size_t ws_bytes, void *stream) {
  return compute_impl(h, N, d_pos, d_type, box, d_off, d_idx, d_shift, d_rev, nnz, d_E, d_Ei, d_F, d_virial, d_ws, ws_bytes,
                      stream, nullptr);
}

static int grade_impl(mtp_handle *h, int64_t N, const double *d_pos, const int32_t *d_type, const double *box,
                      const int64_t *d_off, const int32_t *d_idx, const int8_t *d_shift, int64_t nnz,
                      const double *d_Ainv, int mode, double *d_gamma_atom, double *d_gamma_cfg, double *d_Bsum,
                      double *d_B, void *d_ws, size_t ws_bytes, void *stream, int64_t row_lo = 0, int64_t row_hi = -1) {
  // [row_lo, row_hi): as in compute_impl; gamma_atom and B stay indexed by atom
  if (!h) return MTP_EINVAL;
  const bool window = row_hi >= 0;
  if (!window) { row_lo = 0; row_hi = N; }
  if (row_lo < 0 || row_hi < row_lo || row_hi > N) return fail(h, MTP_EINVAL, "row window outside [0, n_atoms]");
  if (d_off) d_off -= row_lo;
  if (!box || !d_Ainv || mode < 0 || mode > 2 || (N > 0 && (!d_pos || !d_type || !d_off)) || (nnz > 0 && !d_idx) ||
      (mode != 1 && N > 0 && !d_gamma_atom) || (mode != 0 && !d_gamma_cfg))
    return fail(h, MTP_EINVAL, "mtp_grade: null or inconsistent argument");
  cudaStream_t st = (cudaStream_t)stream;
  Plan pl;
  int rc = make_plan(h, N, nnz, 1, 0, pl, -1, window ? row_hi - row_lo : -1);
  if (rc != MTP_OK) return fail(h, rc, "bad sizes");
  const size_t base = align_up((size_t)(uintptr_t)d_ws) - (size_t)(uintptr_t)d_ws;
  // one extra n_basis vector at the end holds sum_i B when the caller does not want it
  const size_t need = pl.total + base + align_up((size_t)h->n_basis * 8);
  if (!d_ws || ws_bytes < need) return fail(h, MTP_ESIZE, "workspace too small");
  PairArgs pa;
  rc = box_setup(h, box, d_shift == nullptr && nnz > 0, h->r_cut, pa);
  if (rc != MTP_OK) return rc;
  char *ws = (char *)d_ws + base;
  double *pos4 = (double *)(ws + pl.o_pos4), *Ei = (double *)(ws + pl.o_Ei), *M = (double *)(ws + pl.o_M);
  double *G = (double *)(ws + pl.o_G), *Bt = (double *)(ws + pl.o_B);      // Bt: tiled [tiles][n_basis][128] of one chunk
  double *Bsum = d_Bsum ? d_Bsum : (double *)(ws + pl.total);
  if (mode != 0 || d_Bsum) CU(h, launch_zero(Bsum, h->n_basis, st));
  if (N > 0) {
    CU(h, launch_pack(d_pos, d_type, (int)N, pos4, st));
    int *idxp = (int *)(ws + pl.o_idxp);
    unsigned *jrange = (unsigned *)(ws + pl.o_jr);
    fill_pair_args(h, pa, pos4, d_off, d_shift ? idxp : d_idx, d_shift);
    pa.n_rows = h->n_basic;
    pa.idx_rel = d_shift ? 1 : 0;
    pa.idx_cap = d_shift ? pl.cap : nnz;
    K2Io io{pos4, M, G, Ei, nullptr, 0, 0, 0, N, (double *)(ws + pl.o_S), (double *)(ws + pl.o_Sbar)};
    for (int c = 0; c < pl.n_chunks; ++c) {
      pa.c0 = (int)(row_lo + c * pl.C); pa.c1 = (int)std::min<int64_t>(row_hi, row_lo + (c + 1) * pl.C);
      if (nnz > 0)
        CU(h, launch_pack_pairs_chunk((const long long *)d_off, pa.c0, pa.c1, d_idx, (const signed char *)d_shift, N, pl.cap,
                                      d_shift ? idxp : nullptr, h->d_flag, jrange, st));
      pa.M = M; pa.kmap = pl.sliced ? h->d_kmapS : h->d_kmapF;
      TIMED(h, CLS_MOMENTS, st, (pl.sliced ? h->pl->moments_s(pa, st) : h->pl->moments(pa, pl.P, st)));
      io.c0 = pa.c0; io.c1 = pa.c1;
      io.B = Bt;
      rc = run_k2(h, io, st);
      if (rc != MTP_OK) return rc;
      const int64_t nc = pa.c1 - pa.c0;
      if (mode != 1) TIMED(h, CLS_GRADE, st, launch_grade(Bt, d_Ainv, nc, h->n_basis, d_gamma_atom + pa.c0, st));
      if (mode != 0 || d_Bsum) CU(h, launch_colsum(Bt, nc, h->n_basis, Bsum, st));
      if (d_B) CU(h, launch_untile(Bt, h->n_basis, nc, d_B + (size_t)pa.c0 * h->n_basis, h->n_basis, 1, st));   // [atom][alpha] for the caller
    }
  }
  if (mode != 0) CU(h, launch_grade_cfg(Bsum, d_Ainv, h->n_basis, nullptr, d_gamma_cfg, st));
  return MTP_OK;
}

extern "C" int mtp_grade(mtp_handle *h, int64_t N, const double *d_pos, const int32_t *d_type, const double *box,
                         const int64_t *d_off, const int32_t *d_idx, const int8_t *d_shift, int64_t nnz,
                         const double *d_Ainv, int mode, double *d_gamma_atom, double *d_gamma_cfg, double *d_Bsum,
                         double *d_B, void *d_ws, size_t ws_bytes, void *stream) {
  return grade_impl(h, N, d_pos, d_type, box, d_off, d_idx, d_shift, nnz, d_Ainv, mode, d_gamma_atom, d_gamma_cfg, d_Bsum, d_B,
                    d_ws, ws_bytes, stream);
}

// ---- small systems: the whole call as one CUDA graph (the small-system variant exists because a
// handful of launches of a few microseconds each dominate below ~10^4 atoms) ---------------------------------------
struct mtp_graph {
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  mtp_handle *h = nullptr;
};

extern "C" int mtp_graph_capture(mtp_handle *h, int64_t N, const double *d_pos, const int32_t *d_type, const double *box,
                                 const int64_t *d_off, const int32_t *d_idx, const int8_t *d_shift, const int32_t *d_rev,
                                 int64_t nnz, double *d_E, double *d_Ei, double *d_F, double *d_virial, void *d_ws,
                                 size_t ws_bytes, mtp_graph **out) {
  if (!h) return MTP_EINVAL;
  if (!out) return fail(h, MTP_EINVAL, "mtp_graph_capture: null argument");
  *out = nullptr;
  cudaStream_t st = nullptr;
  CU(h, cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
  const int saved_profile = h->profile;
  h->profile = 0;                              // timing events cannot be read back from a graph
  cudaError_t e = cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal);
  int rc = MTP_OK;
  cudaGraph_t graph = nullptr;
  if (e == cudaSuccess) {
    rc = compute_impl(h, N, d_pos, d_type, box, d_off, d_idx, d_shift, d_rev, nnz, d_E, d_Ei, d_F, d_virial, d_ws, ws_bytes, st, nullptr);
    e = cudaStreamEndCapture(st, &graph);      // also ends a capture the call invalidated
  }
  h->profile = saved_profile;
  cudaStreamDestroy(st);
  if (rc != MTP_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
  if (e != cudaSuccess || !graph) { cudaGetLastError(); return cuda_fail(h, e, "mtp_graph_capture"); }
  mtp_graph *g = new (std::nothrow) mtp_graph;
  if (!g) { cudaGraphDestroy(graph); return fail(h, MTP_ENOMEM, "out of host memory"); }
  g->graph = graph; g->h = h;
  e = cudaGraphInstantiate(&g->exec, graph, 0);
  if (e != cudaSuccess) { cudaGraphDestroy(graph); delete g; return cuda_fail(h, e, "cudaGraphInstantiate"); }
  *out = g;
  return MTP_OK;
}

extern "C" int mtp_graph_launch(mtp_graph *g, void *stream) {
  if (!g || !g->exec) return MTP_EINVAL;
  cudaError_t e = cudaGraphLaunch(g->exec, (cudaStream_t)stream);
  if (e != cudaSuccess) return cuda_fail(g->h, e, "cudaGraphLaunch");
  return MTP_OK;
}

extern "C" int mtp_graph_destroy(mtp_graph *g) {
  if (!g) return MTP_OK;
  if (g->exec) cudaGraphExecDestroy(g->exec);
  if (g->graph) cudaGraphDestroy(g->graph);
  delete g;
  return MTP_OK;
}

// ---- one rank's share of a sharded evaluation ----------------------------------------
extern "C" int mtp_rows_workspace_bytes(const mtp_handle *h, int64_t n_atoms, int64_t n_rows, int64_t nnz, int want_grade,
                                        size_t *out) {
  if (!h || !out || n_rows < 0) return MTP_EINVAL;
  Plan pl;
  int rc = make_plan(h, n_atoms, nnz, want_grade, /*has_rev=*/0, pl, -1, n_rows);
  if (rc != MTP_OK) return rc;
  *out = pl.total + 512 + (want_grade ? align_up((size_t)h->n_basis * 8) : 0);
  return MTP_OK;
}

extern "C" int mtp_compute_rows(mtp_handle *h, int64_t N, const double *d_pos, const int32_t *d_type, const double *box,
                                int64_t row_lo, int64_t row_hi, const int64_t *d_off, const int32_t *d_idx, const int8_t *d_shift,
                                int64_t nnz, double *d_E, double *d_Ei, double *d_F, double *d_virial, void *d_ws,
                                size_t ws_bytes, void *stream) {
  if (!h) return MTP_EINVAL;
  if (row_lo < 0 || row_hi < row_lo) return fail(h, MTP_EINVAL, "row window outside [0, n_atoms]");
  const int saved = h->force_mode;
  if (saved == MTP_FORCE_AUTO) h->force_mode = MTP_FORCE_ATOMIC;
  int rc = compute_impl(h, N, d_pos, d_type, box, d_off, d_idx, d_shift, nullptr, nnz, d_E, d_Ei, d_F, d_virial, d_ws, ws_bytes,
                        stream, nullptr, -1, row_lo, row_hi);
  h->force_mode = saved;
  return rc;
}

extern "C" int mtp_grade_rows(mtp_handle *h, int64_t N, const double *d_pos, const int32_t *d_type, const double *box,
                              int64_t row_lo, int64_t row_hi, const int64_t *d_off, const int32_t *d_idx, const int8_t *d_shift,
                              int64_t nnz, const double *d_Ainv, double *d_gamma_atom, double *d_Bsum, void *d_ws, size_t ws_bytes,
                              void *stream) {
  if (!h) return MTP_EINVAL;
  if (row_lo < 0 || row_hi < row_lo || !d_Bsum) return fail(h, MTP_EINVAL, "mtp_grade_rows: bad argument");
  return grade_impl(h, N, d_pos, d_type, box, d_off, d_idx, d_shift, nnz, d_Ainv, 0, d_gamma_atom, nullptr, d_Bsum, nullptr, d_ws,
                    ws_bytes, stream, row_lo, row_hi);
}

extern "C" int mtp_grade_cfg_from_sum(mtp_handle *h, const double *d_Bsum, const double *d_Ainv, double *d_gamma_cfg, void *stream) {
  if (!h) return MTP_EINVAL;
  if (!d_Bsum || !d_Ainv || !d_gamma_cfg) return fail(h, MTP_EINVAL, "mtp_grade_cfg_from_sum: null argument");
  CU(h, launch_grade_cfg(d_Bsum, d_Ainv, h->n_basis, nullptr, d_gamma_cfg, (cudaStream_t)stream));
  return MTP_OK;
}

// ---- host-buffer end-to-end path ----------------------------------------------------------
extern "C" int mtp_compute_host(mtp_handle *h, int64_t N, const double *pos, const int32_t *type, const double *box,
                                const int64_t *off, const int32_t *idx, const int8_t *shift, const int32_t *rev,
                                int64_t nnz, double *E, double *Ei, double *F, double *virial) {
  if (!h) return MTP_EINVAL;
  if (!box || !E || (N > 0 && (!pos || !type || !off || !F)) || (nnz > 0 && !idx)) return fail(h, MTP_EINVAL, "mtp_compute_host: null argument");
  // Chunks are the unit of the copy / compute pipeline here (the list of chunk c + 1 crosses PCIe while chunk c is
  // evaluated), so the automatic choice is at most 2^18 atoms instead of as few chunks as possible
  struct ChunkGuard {
    mtp_handle *h; int64_t saved;
    ~ChunkGuard() { h->chunk_atoms = saved; }
  } guard{h, h->chunk_atoms};
  if (h->chunk_atoms <= 0 && N > (1 << 18)) {
    const int64_t nc = (N + (1 << 18) - 1) >> 18;
    h->chunk_atoms = ((N + nc - 1) / nc + 31) / 32 * 32;
  }
  // the CSR offsets are on the host here: the per-pair scratch is sized for the largest chunk exactly
  Plan pl;
  int rc = make_plan(h, N, nnz, 0, rev != nullptr, pl);
  if (rc != MTP_OK) return fail(h, rc, "bad sizes");
  int64_t cap = 0;
  for (int c = 0; c < pl.n_chunks; ++c)
    cap = std::max<int64_t>(cap, off[std::min<int64_t>(N, (int64_t)(c + 1) * pl.C)] - off[(int64_t)c * pl.C]);
  rc = make_plan(h, N, nnz, 0, rev != nullptr, pl, cap);
  if (rc != MTP_OK) return fail(h, rc, "bad sizes");
  const size_t wsb = pl.total + 512;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
  const size_t o_pos = take((size_t)N * 24), o_type = take((size_t)N * 4), o_off = take((size_t)(N + 1) * 8);
  const size_t o_idx = take((size_t)nnz * 4), o_shift = take(shift ? (size_t)nnz * 3 : 0), o_rev = take(rev ? (size_t)nnz * 4 : 0);
  const size_t o_out = take((size_t)(7 + N + 3 * N) * 8), o_ws = take(wsb);
  if (o > h->stage_bytes) {
    if (h->stage) cudaFree(h->stage);
    h->stage = nullptr; h->stage_bytes = 0;
    CU(h, cudaMalloc(&h->stage, o));
    h->stage_bytes = o;
  }
  char *d = (char *)h->stage;
  // Two streams: the neighbour list (the bulk of the input: 11 B per pair) is copied chunk by chunk on the copy
  // stream while the compute stream already evaluates the chunks that have arrived.  (Overlap needs pinned host
  // buffers; with pageable memory the copies simply serialise.)
  if (!h->s_copy) {
    CU(h, cudaStreamCreateWithFlags(&h->s_copy, cudaStreamNonBlocking));
    CU(h, cudaStreamCreateWithFlags(&h->s_comp, cudaStreamNonBlocking));
  }
  while ((int)h->ev.size() < pl.n_chunks + 2) {
    cudaEvent_t e = nullptr;
    CU(h, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    h->ev.push_back(e);
  }
  cudaStream_t sc = h->s_copy, st = h->s_comp;
  std::vector<long long> pair0(pl.n_chunks + 1, 0);
  std::vector<cudaEvent_t> ready(h->ev.begin() + 2, h->ev.begin() + 2 + pl.n_chunks);
  if (N > 0) {
    CU(h, cudaMemcpyAsync(d + o_pos, pos, (size_t)N * 24, cudaMemcpyHostToDevice, sc));
    CU(h, cudaMemcpyAsync(d + o_type, type, (size_t)N * 4, cudaMemcpyHostToDevice, sc));
    CU(h, cudaMemcpyAsync(d + o_off, off, (size_t)(N + 1) * 8, cudaMemcpyHostToDevice, sc));
  }
  CU(h, cudaEventRecord(h->ev[0], sc));
  for (int c = 0; c < pl.n_chunks; ++c) {
    const long long p0 = off[(int64_t)c * pl.C], p1 = off[std::min<int64_t>(N, (int64_t)(c + 1) * pl.C)];
    pair0[c] = p0; pair0[c + 1] = p1;
    if (p1 > p0) {
      CU(h, cudaMemcpyAsync(d + o_idx + 4 * p0, idx + p0, (size_t)(p1 - p0) * 4, cudaMemcpyHostToDevice, sc));
      if (shift) CU(h, cudaMemcpyAsync(d + o_shift + 3 * p0, shift + 3 * p0, (size_t)(p1 - p0) * 3, cudaMemcpyHostToDevice, sc));
    }
    CU(h, cudaEventRecord(ready[c], sc));
    if (c == 0) {      // the reverse index is needed by the first chunk's force assembly: it travels while chunk 0 is evaluated
      if (rev && nnz > 0) CU(h, cudaMemcpyAsync(d + o_rev, rev, (size_t)nnz * 4, cudaMemcpyHostToDevice, sc));
      CU(h, cudaEventRecord(h->ev[1], sc));
    }
  }
  if (pl.n_chunks == 0) CU(h, cudaEventRecord(h->ev[1], sc));
  CU(h, cudaStreamWaitEvent(st, h->ev[0], 0));
  HostPipe pipe;
  pipe.chunk_ready = &ready; pipe.chunk_pair0 = &pair0; pipe.rev_ready = h->ev[1];
  double *dE = (double *)(d + o_out), *dW = dE + 1, *dEi = dE + 7, *dF = dEi + N;
  rc = compute_impl(h, N, (double *)(d + o_pos), (int32_t *)(d + o_type), box, (int64_t *)(d + o_off),
                    (int32_t *)(d + o_idx), shift ? (int8_t *)(d + o_shift) : nullptr,
                    rev ? (int32_t *)(d + o_rev) : nullptr, nnz, dE, dEi, dF, dW, d + o_ws, wsb, st, N > 0 ? &pipe : nullptr, cap);
  if (rc != MTP_OK) { cudaStreamSynchronize(sc); cudaStreamSynchronize(st); return rc; }
  if (N == 0) CU(h, cudaStreamWaitEvent(st, h->ev[1], 0));
  CU(h, cudaMemcpyAsync(E, dE, 8, cudaMemcpyDeviceToHost, st));
  if (virial) CU(h, cudaMemcpyAsync(virial, dW, 48, cudaMemcpyDeviceToHost, st));
  if (Ei && N > 0) CU(h, cudaMemcpyAsync(Ei, dEi, (size_t)N * 8, cudaMemcpyDeviceToHost, st));
  if (N > 0) CU(h, cudaMemcpyAsync(F, dF, (size_t)N * 24, cudaMemcpyDeviceToHost, st));
  CU(h, cudaStreamSynchronize(st));
  return MTP_OK;
}

// ---- device neighbour list, MD loop --------------------------------------------------------
extern "C" int mtp_neighbors_workspace_bytes(int64_t n_atoms, size_t *out) {
  if (n_atoms < 0 || !out) return MTP_EINVAL;
  *out = nb_workspace_bytes(n_atoms);
  return MTP_OK;
}

extern "C" int mtp_neighbors_build(int64_t N, const double *d_pos, const double *box, double r_list, int64_t capacity,
                                   int64_t *d_off, int32_t *d_idx, int8_t *d_shift, int32_t *d_rev, int64_t *d_info,
                                   void *d_ws, size_t ws_bytes, void *stream) {
  if (N < 0 || N > (1LL << 27) || !box || !d_off || !d_info || capacity < 0 || (N > 0 && !d_pos) ||
      (capacity > 0 && (!d_idx || !d_shift)) || capacity > 0x7fffffffLL)
    return MTP_EINVAL;
  if (!d_ws || ws_bytes < nb_workspace_bytes(N)) return MTP_ESIZE;
  NbGrid g;
  if (!nb_grid(box, r_list, N, g)) return MTP_EBOX;
  char *ws = (char *)d_ws;
  ws += (256 - ((uintptr_t)ws & 255)) & 255;
  cudaError_t e = launch_neighbors_build(g, N, d_pos, r_list, capacity, (long long *)d_off, d_idx, (signed char *)d_shift, d_rev,
                                         (long long *)d_info, 0, ws, (cudaStream_t)stream);
  return e == cudaSuccess ? MTP_OK : MTP_ECUDA;
}

namespace {
// LAMMPS "metal" units: eV, Angstrom, ps, g/mol.  a [A/ps^2] = F [eV/A] / m [g/mol] x kFtm2v
constexpr double kFtm2v = 1.602176634e-19 / 1.66053906660e-27 * 1e-4;      // 9648.533...
struct MdLayout { size_t off, idx, shift, rev, info, imass, mass, ke, gamma, gmax, nbws, ws, total; };
MdLayout md_layout(const mtp_handle *h, int64_t N, int64_t cap, size_t compute_ws, bool policy = false) {
  MdLayout L;
  size_t o = 0;
  auto take = [&](size_t b) { size_t at = o; o = align_up(o + b); return at; };
  L.off = take((size_t)(N + 1) * 8); L.idx = take((size_t)cap * 4); L.shift = take((size_t)cap * 3); L.rev = take((size_t)cap * 4);
  L.info = take(16); L.imass = take((size_t)h->S * 8); L.mass = take((size_t)h->S * 8); L.ke = take((size_t)N * 8);
  L.gamma = take(policy ? (size_t)N * 8 : 0); L.gmax = take(policy ? 8 : 0);
  L.nbws = take(nb_workspace_bytes(N)); L.ws = take(compute_ws);
  L.total = o;
  return L;
}
}  // namespace

extern "C" int mtp_md_workspace_bytes(const mtp_handle *h, int64_t n_atoms, int64_t capacity, size_t *out) {
  if (!h || !out || n_atoms < 0 || capacity < 0) return MTP_EINVAL;
  size_t cw = 0;
  int rc = mtp_workspace_bytes(h, n_atoms, capacity, 0, &cw);
  if (rc != MTP_OK) return rc;
  *out = md_layout(h, n_atoms, capacity, cw).total + 512;
  return MTP_OK;
}

namespace {
// what the active-learning policy needs on top of the plain loop (mtp_md_run_al)
struct MdPolicy {
  const mtp_al_policy *p = nullptr;
  const double *d_Ainv = nullptr;
  double *d_gamma_atom = nullptr;          // [N] or nullptr (then a workspace array)
  double *d_selected = nullptr;            // [max_selected][N][3] or nullptr
  int64_t *sel_step = nullptr;             // host [max_selected]
  double *sel_grade = nullptr;             // host [max_selected]
  int64_t *out = nullptr;                  // host [4]: steps done, configurations selected, grade evaluations, 1 = stopped at the break threshold
  double *max_grade = nullptr;             // host [1]: largest grade seen
};

int md_impl(mtp_handle *h, int64_t N, double *d_pos, double *d_vel, const int32_t *d_type, const double *box, const double *mass,
            double dt, int64_t n_steps, int32_t rebuild_every, double skin, int64_t capacity, double *d_E, double *d_Ei, double *d_F,
            double *d_virial, int64_t *d_info, void *d_ws, size_t ws_bytes, void *stream, const MdPolicy *al) {
  if (!h) return MTP_EINVAL;
  if (N <= 0 || !d_pos || !d_vel || !d_type || !box || !mass || !(dt > 0) || n_steps < 0 || rebuild_every < 1 || !(skin >= 0) ||
      capacity <= 0 || capacity > 0x7fffffffLL || !d_E || !d_F || !d_info)
    return fail(h, MTP_EINVAL, "mtp_md_run: bad argument");
  if (al && (!al->p || !al->d_Ainv || !al->out || al->p->grade_every < 1 || al->p->mode < 0 || al->p->mode > 1 || al->p->max_selected < 0 ||
             (al->p->max_selected > 0 && (!al->sel_step || !al->sel_grade))))
    return fail(h, MTP_EINVAL, "mtp_md_run_al: bad policy argument");
  for (int s = 0; s < h->S; ++s) if (!(mass[s] > 0)) return fail(h, MTP_EINVAL, "mtp_md_run: masses must be positive");
  cudaStream_t st = (cudaStream_t)stream;
  size_t cw = 0, gw = 0;
  int rc = mtp_workspace_bytes(h, N, capacity, 0, &cw);
  if (rc == MTP_OK && al) rc = mtp_workspace_bytes(h, N, capacity, 1, &gw);
  if (rc != MTP_OK) return rc;
  const MdLayout L = md_layout(h, N, capacity, std::max(cw, gw), al != nullptr);
  const size_t base = align_up((size_t)(uintptr_t)d_ws) - (size_t)(uintptr_t)d_ws;
  if (!d_ws || ws_bytes < L.total + base) return fail(h, MTP_ESIZE, "workspace too small (mtp_md_workspace_bytes)");
  char *ws = (char *)d_ws + base;
  int64_t *off = (int64_t *)(ws + L.off);
  int32_t *idx = (int32_t *)(ws + L.idx), *rev = (int32_t *)(ws + L.rev);
  int8_t *shift = (int8_t *)(ws + L.shift);
  double *imass = (double *)(ws + L.imass), *dmass = (double *)(ws + L.mass), *ke = (double *)(ws + L.ke);
  const double r_list = h->r_cut + skin;
  NbGrid g;
  if (!nb_grid(box, r_list, N, g)) return fail(h, MTP_EBOX, "singular box");
  std::vector<double> im(h->S);
  for (int s = 0; s < h->S; ++s) im[s] = 1.0 / mass[s];
  CU(h, cudaMemcpyAsync(imass, im.data(), (size_t)h->S * 8, cudaMemcpyHostToDevice, st));
  CU(h, cudaMemcpyAsync(dmass, mass, (size_t)h->S * 8, cudaMemcpyHostToDevice, st));
  CU(h, cudaStreamSynchronize(st));           // the two host arrays above are the caller's / this frame's
  CU(h, cudaMemsetAsync(d_info, 0, 16, st));
  auto build = [&]() -> int {                 // atoms back into the box, then the list at r_cut + skin (entries beyond r_cut
    CU(h, launch_wrap(g, (int)N, d_pos, st)); // contribute exactly nothing: reading G3)
    CU(h, launch_neighbors_build(g, N, d_pos, r_list, capacity, (long long *)off, idx, (signed char *)shift, rev, (long long *)d_info, 1,
                                 ws + L.nbws, st));
    return MTP_OK;
  };
  auto forces = [&]() {
    return compute_impl(h, N, d_pos, d_type, box, off, idx, shift, rev, capacity, d_E, d_Ei, d_F, d_virial, ws + L.ws, cw, st, nullptr);
  };
  // grades every X steps; above the selection threshold the configuration is kept, above the break
  // threshold the run stops.  The decision is the host's, so each evaluation ends with a 8-byte read and a
  // synchronisation.  0 = go on, 1 = stop, < 0 = error.
  int64_t n_sel = 0, n_eval = 0;
  double seen_max = 0.0;
  auto policy = [&](int64_t step) -> int {
    double *gamma = al->d_gamma_atom ? al->d_gamma_atom : (double *)(ws + L.gamma);
    double *gmax = (double *)(ws + L.gmax);
    int r = grade_impl(h, N, d_pos, d_type, box, off, idx, shift, capacity, al->d_Ainv, al->p->mode == 0 ? 0 : 1, gamma, gmax,
                       nullptr, nullptr, ws + L.ws, std::max(cw, gw), st);
    if (r != MTP_OK) return r;
    if (al->p->mode == 0) CU(h, launch_max_nonneg(gamma, N, gmax, st));       // neighbourhood mode: the largest per-atom grade
    double m = 0.0;
    CU(h, cudaMemcpyAsync(&m, gmax, 8, cudaMemcpyDeviceToHost, st));
    CU(h, cudaStreamSynchronize(st));
    ++n_eval;
    seen_max = std::max(seen_max, m);
    if (m > al->p->select_threshold && n_sel < al->p->max_selected) {
      if (al->d_selected) CU(h, cudaMemcpyAsync(al->d_selected + (size_t)n_sel * 3 * N, d_pos, (size_t)N * 24, cudaMemcpyDeviceToDevice, st));
      al->sel_step[n_sel] = step; al->sel_grade[n_sel] = m;
      ++n_sel;
    }
    return m > al->p->break_threshold ? 1 : 0;
  };
  const int saved_mode = h->force_mode, saved_skin = h->skin_list;
  if (h->force_mode == MTP_FORCE_AUTO) h->force_mode = MTP_FORCE_GATHER;      // the list comes with its reverse index
  if (skin > 0) h->skin_list = 1;                                             // pairs between R_cut and R_cut + skin are skipped, not multiplied by 0
  rc = build();
  if (rc == MTP_OK) rc = forces();
  int64_t done = 0;
  int stop = 0;
  if (rc == MTP_OK && al) { stop = policy(0); if (stop < 0) rc = stop; }
  const double half = 0.5 * dt * kFtm2v;
  for (int64_t s = 1; s <= n_steps && rc == MTP_OK && stop == 0; ++s) {
    cudaError_t e = launch_vv((int)N, d_pos, d_vel, d_F, d_type, imass, half, dt, 1, st);      // v(t + dt/2), x(t + dt)
    if (e != cudaSuccess) { rc = cuda_fail(h, e, "launch_vv"); break; }
    if (s % rebuild_every == 0) rc = build();
    if (rc == MTP_OK) rc = forces();                                                            // F(t + dt)
    if (rc != MTP_OK) break;
    e = launch_vv((int)N, d_pos, d_vel, d_F, d_type, imass, half, dt, 0, st);                   // v(t + dt)
    if (e != cudaSuccess) { rc = cuda_fail(h, e, "launch_vv"); break; }
    done = s;
    if (al && s % al->p->grade_every == 0) { stop = policy(s); if (stop < 0) rc = stop; }
  }
  h->force_mode = saved_mode; h->skin_list = saved_skin;
  if (rc != MTP_OK) return rc;
  // kinetic energy sum m v^2 / 2 in eV
  CU(h, launch_ke((int)N, d_vel, d_type, dmass, 0.5 / kFtm2v, ke, st));
  CU(h, launch_reduce(ke, N, 1, 1, d_E + 1, nullptr, st));
  if (al) {
    al->out[0] = done; al->out[1] = n_sel; al->out[2] = n_eval; al->out[3] = stop > 0 ? 1 : 0;
    if (al->max_grade) *al->max_grade = seen_max;
  }
  return MTP_OK;
}
}  // namespace

extern "C" int mtp_md_run(mtp_handle *h, int64_t N, double *d_pos, double *d_vel, const int32_t *d_type, const double *box,
                          const double *mass, double dt, int64_t n_steps, int32_t rebuild_every, double skin, int64_t capacity,
                          double *d_E, double *d_Ei, double *d_F, double *d_virial, int64_t *d_info, void *d_ws, size_t ws_bytes,
                          void *stream) {
  return md_impl(h, N, d_pos, d_vel, d_type, box, mass, dt, n_steps, rebuild_every, skin, capacity, d_E, d_Ei, d_F, d_virial, d_info,
                 d_ws, ws_bytes, stream, nullptr);
}

extern "C" int mtp_md_al_workspace_bytes(const mtp_handle *h, int64_t n_atoms, int64_t capacity, size_t *out) {
  if (!h || !out || n_atoms < 0 || capacity < 0) return MTP_EINVAL;
  size_t cw = 0, gw = 0;
  int rc = mtp_workspace_bytes(h, n_atoms, capacity, 0, &cw);
  if (rc == MTP_OK) rc = mtp_workspace_bytes(h, n_atoms, capacity, 1, &gw);
  if (rc != MTP_OK) return rc;
  *out = md_layout(h, n_atoms, capacity, std::max(cw, gw), true).total + 512;
  return MTP_OK;
}

extern "C" int mtp_md_run_al(mtp_handle *h, int64_t N, double *d_pos, double *d_vel, const int32_t *d_type, const double *box,
                             const double *mass, double dt, int64_t n_steps, int32_t rebuild_every, double skin, int64_t capacity,
                             const double *d_Ainv, const mtp_al_policy *policy, double *d_E, double *d_Ei, double *d_F,
                             double *d_virial, int64_t *d_info, double *d_gamma_atom, double *d_selected, int64_t *sel_step,
                             double *sel_grade, int64_t *out, double *max_grade, void *d_ws, size_t ws_bytes, void *stream) {
  MdPolicy al;
  al.p = policy; al.d_Ainv = d_Ainv; al.d_gamma_atom = d_gamma_atom; al.d_selected = d_selected; al.sel_step = sel_step;
  al.sel_grade = sel_grade; al.out = out; al.max_grade = max_grade;
  return md_impl(h, N, d_pos, d_vel, d_type, box, mass, dt, n_steps, rebuild_every, skin, capacity, d_E, d_Ei, d_F, d_virial, d_info,
                 d_ws, ws_bytes, stream, &al);
}

// Host positions in, host forces out: the neighbour list never crosses PCIe (it is built on the device at R_cut).
extern "C" int mtp_compute_host_pos(mtp_handle *h, int64_t N, const double *pos, const int32_t *type, const double *box,
                                    double *E, double *Ei, double *F, double *virial, int64_t *nnz_out) {
  if (!h) return MTP_EINVAL;
  if (N <= 0 || !pos || !type || !box || !E || !F) return fail(h, MTP_EINVAL, "mtp_compute_host_pos: bad argument");
  NbGrid g;
  if (!nb_grid(box, h->r_cut, N, g)) return fail(h, MTP_EBOX, "singular box");
  if (!h->s_comp) {
    CU(h, cudaStreamCreateWithFlags(&h->s_copy, cudaStreamNonBlocking));
    CU(h, cudaStreamCreateWithFlags(&h->s_comp, cudaStreamNonBlocking));
  }
  cudaStream_t st = h->s_comp;
  const int saved_mode = h->force_mode;
  for (int attempt = 0; attempt < 3; ++attempt) {
    const int64_t cap = h->nb_capacity;
    size_t cw = 0;
    int rc = mtp_workspace_bytes(h, N, std::max<int64_t>(cap, 1), 0, &cw);
    if (rc != MTP_OK) return rc;
    size_t o = 0;
    auto take = [&](size_t b) { size_t at = o; o = align_up(o + b); return at; };
    const size_t o_pos = take((size_t)N * 24), o_type = take((size_t)N * 4), o_off = take((size_t)(N + 1) * 8);
    const size_t o_idx = take((size_t)cap * 4), o_shift = take((size_t)cap * 3), o_rev = take((size_t)cap * 4), o_info = take(16);
    const size_t o_out = take((size_t)(7 + 4 * N) * 8), o_nbws = take(nb_workspace_bytes(N)), o_ws = take(cw);
    if (o > h->stage_nb_bytes) {
      if (h->stage_nb) cudaFree(h->stage_nb);
      h->stage_nb = nullptr; h->stage_nb_bytes = 0;
      CU(h, cudaMalloc(&h->stage_nb, o));
      h->stage_nb_bytes = o;
    }
    char *d = (char *)h->stage_nb;
    CU(h, cudaMemcpyAsync(d + o_pos, pos, (size_t)N * 24, cudaMemcpyHostToDevice, st));
    CU(h, cudaMemcpyAsync(d + o_type, type, (size_t)N * 4, cudaMemcpyHostToDevice, st));
    CU(h, launch_neighbors_build(g, N, (double *)(d + o_pos), h->r_cut, cap, (long long *)(d + o_off), (int *)(d + o_idx),
                                 (signed char *)(d + o_shift), (int *)(d + o_rev), (long long *)(d + o_info), 0, d + o_nbws, st));
    long long info[2] = {0, 0};
    if (cap > 0) {
      double *dE = (double *)(d + o_out), *dW = dE + 1, *dEi = dE + 7, *dF = dEi + N;
      if (h->force_mode == MTP_FORCE_AUTO) h->force_mode = MTP_FORCE_GATHER;
      rc = compute_impl(h, N, (double *)(d + o_pos), (int32_t *)(d + o_type), box, (int64_t *)(d + o_off), (int32_t *)(d + o_idx),
                        (int8_t *)(d + o_shift), (int32_t *)(d + o_rev), cap, dE, dEi, dF, dW, d + o_ws, cw, st, nullptr);
      h->force_mode = saved_mode;
      if (rc != MTP_OK) { cudaStreamSynchronize(st); return rc; }
      CU(h, cudaMemcpyAsync(E, dE, 8, cudaMemcpyDeviceToHost, st));
      if (virial) CU(h, cudaMemcpyAsync(virial, dW, 48, cudaMemcpyDeviceToHost, st));
      if (Ei) CU(h, cudaMemcpyAsync(Ei, dEi, (size_t)N * 8, cudaMemcpyDeviceToHost, st));
      CU(h, cudaMemcpyAsync(F, dF, (size_t)N * 24, cudaMemcpyDeviceToHost, st));
    }
    CU(h, cudaMemcpyAsync(info, d + o_info, 16, cudaMemcpyDeviceToHost, st));
    CU(h, cudaStreamSynchronize(st));
    if (info[1] != 0) return fail(h, MTP_EUNSUP, "neighbour rows longer than 256 entries");
    if (nnz_out) *nnz_out = info[0];
    if (info[0] <= cap && cap > 0) return MTP_OK;
    if (info[0] == 0) {                          // no pairs at all: E_i = xi0, F = 0 -- run the plain path with an empty list
      h->nb_capacity = 1;
      if (cap > 0) return MTP_OK;
      continue;
    }
    h->nb_capacity = info[0] + info[0] / 16 + 1024;        // first call, or the list outgrew the buffers: size them and redo
  }
  return fail(h, MTP_ESIZE, "neighbour list kept outgrowing its buffers");
}

// ---- diagnostics ------------------------------------------------------------------------------
extern "C" int mtp_debug_moments(mtp_handle *h, int64_t N, const double *d_pos, const int32_t *d_type,
                                 const double *box, const int64_t *d_off, const int32_t *d_idx, const int8_t *d_shift,
                                 double *d_M, double *d_G, double *d_B, void *d_ws, size_t ws_bytes, void *stream) {
  if (!h || !box || N <= 0 || !d_pos || !d_type || !d_off || !d_idx) return MTP_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t saved = h->chunk_atoms;
  h->chunk_atoms = N;                       // single chunk so that M, G hold every atom
  Plan pl;
  int rc = make_plan(h, N, 0, 1, 0, pl);    // sized like a grade call: the plan then has room for the tiled B
  h->chunk_atoms = saved;
  if (rc != MTP_OK) return rc;
  const size_t base = align_up((size_t)(uintptr_t)d_ws) - (size_t)(uintptr_t)d_ws;
  if (!d_ws || ws_bytes < pl.total + base) return fail(h, MTP_ESIZE, "workspace too small (size it with want_grade = 1)");
  PairArgs pa;
  rc = box_setup(h, box, d_shift == nullptr, h->r_cut, pa);
  if (rc != MTP_OK) return rc;
  char *ws = (char *)d_ws + base;
  double *pos4 = (double *)(ws + pl.o_pos4), *Ei = (double *)(ws + pl.o_Ei), *M = (double *)(ws + pl.o_M), *G = (double *)(ws + pl.o_G);
  double *Bt = (double *)(ws + pl.o_B);
  CU(h, launch_pack(d_pos, d_type, (int)N, pos4, st));
  int *tmp_idxp = nullptr;                  // diagnostics only: this entry point has no nnz argument
  if (d_shift) {
    long long nnz = 0;
    CU(h, cudaMemcpyAsync(&nnz, d_off + N, 8, cudaMemcpyDeviceToHost, st));
    CU(h, cudaStreamSynchronize(st));
    CU(h, cudaMalloc((void **)&tmp_idxp, (size_t)std::max<long long>(nnz, 1) * 4));
    cudaError_t e = launch_pack_pairs_chunk((const long long *)d_off, 0, (int)N, d_idx, (const signed char *)d_shift, N, nnz, tmp_idxp,
                                            h->d_flag, (unsigned *)(ws + pl.o_jr), st);
    if (e != cudaSuccess) { cudaFree(tmp_idxp); return cuda_fail(h, e, "launch_pack_pairs_chunk"); }
  }
  fill_pair_args(h, pa, pos4, d_off, tmp_idxp ? tmp_idxp : d_idx, d_shift);
  pa.idx_rel = 0;                            // one chunk starting at atom 0: relative = absolute
  pa.n_rows = h->n_basic; pa.c0 = 0; pa.c1 = (int)N; pa.M = M; pa.kmap = pl.sliced ? h->d_kmapS : h->d_kmapF;
  {
    cudaError_t e = pl.sliced ? h->pl->moments_s(pa, st) : h->pl->moments(pa, pl.P, st);
    if (tmp_idxp) { cudaStreamSynchronize(st); cudaFree(tmp_idxp); }
    if (e != cudaSuccess) return cuda_fail(h, e, "moments");
  }
  // B is exported, so every basis value is stored (no leaf elision)
  K2Io io{pos4, M, G, Ei, Bt, 0, (int)N, 1, N, (double *)(ws + pl.o_S), (double *)(ws + pl.o_Sbar)};
  rc = run_k2(h, io, st);
  if (rc != MTP_OK) return rc;
  // outputs: M, G as [n_basic][N] (component-major), B as [N][n_basis]
  if (d_M) CU(h, launch_untile(M, h->n_basic, N, d_M, N, 0, st));
  if (d_G) CU(h, launch_untile(G, h->n_basic, N, d_G, N, 0, st));
  if (d_B) CU(h, launch_untile(Bt, h->n_basis, N, d_B, h->n_basis, 1, st));
  return MTP_OK;
}

extern "C" int mtp_peak_dfma(int64_t iters, double *d_sink, double *out_flops, void *stream) {
  if (iters <= 0 || !d_sink) return MTP_EINVAL;
  return launch_peak_dfma(iters, d_sink, out_flops, (cudaStream_t)stream) == cudaSuccess ? MTP_OK : MTP_ECUDA;
}

// Useful flops (FMA = 2), every quantity counted once, recomputation not counted -- DESIGN.md section 6:
//   K1 per pair  30 + 16 n_mu + 2 C(nu_max + 3, 3) + 2 n_basic      (geometry, radial functions, monomials, moments)
//   K3 per pair  30 + 16 n_mu + 8 n_basic                            (radial derivatives, value + gradient of sum_mu f_mu P_mu)
//   K2 per atom  6 n_prod + 2 n_basis                                (forward 2 / op, adjoint 4 / op, energy)
//   K5 per atom  2 n_basis^2
// flop_per_pair[0] = K1, [1] = K3.
extern "C" int mtp_cost_model(const mtp_handle *h, double *flop_per_pair, double *flop_per_atom_tree,
                              double *flop_per_atom_grade) {
  if (!h) return MTP_EINVAL;
  const int numax = rt_numax(h->pl->lev, 0);
  const double monos = (numax + 1.0) * (numax + 2.0) * (numax + 3.0) / 6.0;
  if (flop_per_pair) {
    flop_per_pair[0] = 30.0 + 16.0 * h->nmu + 2.0 * monos + 2.0 * h->n_basic;
    flop_per_pair[1] = 30.0 + 16.0 * h->nmu + 8.0 * h->n_basic;
  }
  if (flop_per_atom_tree) *flop_per_atom_tree = 6.0 * (double)h->n_prod + 2.0 * h->n_basis;
  if (flop_per_atom_grade) *flop_per_atom_grade = 2.0 * (double)h->n_basis * h->n_basis;
  return MTP_OK;
}

// Host-only: the register program mtp_create would run for this table (whole table only; kind 0 = energy + adjoint,
// 1 = basis values), for emulation in the tests.  prog receives up to cap instructions of 7 int32 each
// (op, d, a, b, c, k, x -- tree_codegen.h), consts up to ccap doubles; info = {instructions, constants, registers, slots}.
extern "C" int mtp_k2_program(const mtp_params *p, int kind, int32_t *prog, int64_t cap, double *consts, int64_t ccap,
                              int64_t *info) {
  if (!p || !info || kind < 0 || kind > 1 || !p->xi) return MTP_EINVAL;
  K2Table whole;
  const char *verr = "";
  if (k2_validate(p->n_basic, p->n_nodes, p->n_prod, p->prod, p->n_basis, p->basis_node, &verr) != MTP_OK) return MTP_EINVAL;
  whole.n_basic = p->n_basic; whole.n_nodes = p->n_nodes; whole.prod.assign(p->prod, p->prod + 4 * (size_t)p->n_prod);
  whole.basis_node.assign(p->basis_node, p->basis_node + p->n_basis);
  whole.xi.assign(p->xi, p->xi + p->n_basis);
  K2Gen g;
  std::string err;
  int rc = k2_generate(whole, (K2Kind)kind, kK2Window, kK2Lookahead, g, &err);
  if (rc != MTP_OK) { g_create_error = err; return rc; }
  info[0] = (int64_t)g.prog.size(); info[1] = (int64_t)g.consts.size(); info[2] = g.n_regs; info[3] = g.n_slots;
  if (prog && cap >= (int64_t)g.prog.size()) std::memcpy(prog, g.prog.data(), g.prog.size() * sizeof(K2Inst));
  if (consts && ccap >= (int64_t)g.consts.size() && !g.consts.empty()) std::memcpy(consts, g.consts.data(), g.consts.size() * 8);
  return MTP_OK;
}
