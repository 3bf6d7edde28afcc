// K2 specialised at mtp_create time: the lane programs of tree.h are turned into straight-line CUDA
// source (one code region per wave and row-lane warp, shared-memory operands at immediate offsets,
// multipliers as literals), compiled with NVRTC for sm_100a and loaded through the runtime's library
// API.  Same mapping and same arithmetic order as the interpreter in tree_kernel.cu (atoms across
// lanes, AL = 32, AR atoms per lane, warps = row-lanes), so results are bit-identical; what goes away
// is the per-entry fetch / decode / branch work (~20 instructions per entry -> 2 loads + AR FMAs).
// NVRTC is dlopen'ed: without it (or when a program is too long to be worth compiling) the
// interpreter runs instead -- both are CUDA paths.  BASELINE.json north_star: "forward/adjoint
// contraction kernel with the tree in registers and shared memory".
#include <cuda_runtime.h>
#include <dlfcn.h>

#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "kernels.h"

namespace mtpb {

namespace {
// ---- the few NVRTC entry points we need, resolved at run time
typedef struct _nvrtcProgram *nvrtcProgram;
struct Nvrtc {
  int (*CreateProgram)(nvrtcProgram *, const char *, const char *, int, const char *const *, const char *const *) = nullptr;
  int (*CompileProgram)(nvrtcProgram, int, const char *const *) = nullptr;
  int (*GetCUBINSize)(nvrtcProgram, size_t *) = nullptr;
  int (*GetCUBIN)(nvrtcProgram, char *) = nullptr;
  int (*GetProgramLogSize)(nvrtcProgram, size_t *) = nullptr;
  int (*GetProgramLog)(nvrtcProgram, char *) = nullptr;
  int (*DestroyProgram)(nvrtcProgram *) = nullptr;
  bool ok = false;
};
const Nvrtc &nvrtc() {
  static Nvrtc n = [] {
    Nvrtc r;
    void *h = nullptr;
    for (const char *name : {"libnvrtc.so.12", "libnvrtc.so", "/usr/local/cuda/lib64/libnvrtc.so.12"})
      if ((h = dlopen(name, RTLD_NOW | RTLD_LOCAL))) break;
    if (!h) return r;
    auto sym = [&](const char *s) { return dlsym(h, s); };
    r.CreateProgram = (decltype(r.CreateProgram))sym("nvrtcCreateProgram");
    r.CompileProgram = (decltype(r.CompileProgram))sym("nvrtcCompileProgram");
    r.GetCUBINSize = (decltype(r.GetCUBINSize))sym("nvrtcGetCUBINSize");
    r.GetCUBIN = (decltype(r.GetCUBIN))sym("nvrtcGetCUBIN");
    r.GetProgramLogSize = (decltype(r.GetProgramLogSize))sym("nvrtcGetProgramLogSize");
    r.GetProgramLog = (decltype(r.GetProgramLog))sym("nvrtcGetProgramLog");
    r.DestroyProgram = (decltype(r.DestroyProgram))sym("nvrtcDestroyProgram");
    r.ok = r.CreateProgram && r.CompileProgram && r.GetCUBINSize && r.GetCUBIN && r.DestroyProgram;
    return r;
  }();
  return n;
}

// Kernel frame: prologue / epilogue as in tree_kernel.cu; @FWD@ / @BWD@ receive the generated passes.
const char *kFrame = R"SRC(
struct TreeTerm;
struct TreeArgs {
  const TreeTerm *fprog; const int *fwave; int nfw;
  const TreeTerm *bprog; const int *bwave; int nbw;
  int n_fprog, n_bprog;
  int prog_smem_off;
  const double *xi0;
  const double *adj_init;
  const double *leaf_seed;
  const int *eseed_slot; const double *eseed_val; int n_eseed;
  const int *basis_slot;
  const int *gseed_k; const double *gseed_val; int n_gseed;
  const int *gzero_k; int n_gzero;
  const double *pos4;
  const double *M; double *G; long long ldm;
  double *Ei;
  double *B;
  int n_val, n_adj, n_basic, n_basis;
  int c0, c1;
  int want_adj;
  const int *mload_k;                      // the fields below serve the group sub-programs of a partitioned tree
  const int *cut_row, *cut_vslot, *cut_aslot; int n_cut;
  double *S;
  const double *Sbar;
  int g_accum;
  int write_energy;
};
// four table offsets with one 16-byte load through L1 (the tables are streamed once per atom group: global memory,
// not the constant bank, whose cache is made for reuse -- measured 4.2 ms against 2.8 ms of the straight-line form)
__device__ __forceinline__ uint4 LQ(const uint4 *p) { return __ldg(p); }
#define AR @AR@
#define GRP @GRP@        // 1: group sub-program of a partitioned tree (subset loads, per-atom seeds, G accumulates)
#define NT @NT@
#define AL 32
#define A (AL * AR)
#define R (NT / AL)
#if AR == 2
#define LD(p) (*(const double2 *)(p))
// E0 / G0 open a group / row with a multiply (== fma onto an exact zero, without the zeroing instructions;
// __dmul_rn keeps the compiler from contracting it with a later add)
#define E0(OA, OB) { const double2 X = LD(s0 + OA), Y = LD(vc + OB); ax = __dmul_rn(X.x, Y.x); ay = __dmul_rn(X.y, Y.y); }
#define E(OA, OB) { const double2 X = LD(s0 + OA), Y = LD(vc + OB); ax = fma(X.x, Y.x, ax); ay = fma(X.y, Y.y, ay); }
#define G0(M) { tx = __dmul_rn(M, ax); ty = __dmul_rn(M, ay); }
#define GC(M) { tx = fma(M, ax, tx); ty = fma(M, ay, ty); }
// exact shortcuts: a first factor that is the constant 1 (adj slot 0), a multiplier 1, a row that is the only
// contribution to an adjoint whose initial value I is known here
#define Y0(OB) { const double2 Y = LD(vc + OB); ax = Y.x; ay = Y.y; }
#define Y1(OB) { const double2 Y = LD(vc + OB); ax += Y.x; ay += Y.y; }
#define G1() { tx = ax; ty = ay; }
#define RS(D) { *(double2 *)(ac + D) = make_double2(tx, ty); }
#define RI(D, I) { *(double2 *)(ac + D) = make_double2(I + tx, I + ty); }
#define RV(D) { *(double2 *)(vw + D) = make_double2(tx, ty); }
#define RL(S) { ex = fma(S, tx, ex); ey = fma(S, ty, ey); }
#define RA(D) { double2 o = LD(ac + D); o.x += tx; o.y += ty; *(double2 *)(ac + D) = o; }
// rows of G: ldm is a multiple of 64 (api.cu make_plan) and a lane's two atoms sit on 16 bytes, so a row is one
// unpredicated 16-byte store at a 32-bit index (the columns of atoms past the chunk's end are padding)
#define GP(K) ((double2 *)(Gcol + (unsigned)(K) * ldm32))
#define RGA(K) { double2 *gp = GP(K); double2 o = *gp; o.x += tx; o.y += ty; *gp = o; }   // later piece of a split row
#if GRP
#define RG(K) { double2 *gp = GP(K); double2 o = make_double2(tx, ty); if (ga) { const double2 p = *gp; o.x = p.x + tx; o.y = p.y + ty; } *gp = o; }
#else
#define RG(K) { *GP(K) = make_double2(tx, ty); }
#endif
#else
#define LD(p) (*(const double *)(p))
#define E0(OA, OB) { ax = __dmul_rn(LD(s0 + OA), LD(vc + OB)); }
#define E(OA, OB) { ax = fma(LD(s0 + OA), LD(vc + OB), ax); }
#define G0(M) { tx = __dmul_rn(M, ax); }
#define GC(M) { tx = fma(M, ax, tx); }
#define Y0(OB) { ax = LD(vc + OB); }
#define Y1(OB) { ax += LD(vc + OB); }
#define G1() { tx = ax; }
#define RS(D) { *(double *)(ac + D) = tx; }
#define RI(D, I) { *(double *)(ac + D) = I + tx; }
#define RV(D) { *(double *)(vw + D) = tx; }
#define RL(S) { ex = fma(S, tx, ex); }
#define RA(D) { *(double *)(ac + D) += tx; }
#define RGA(K) { double *gp = Gcol + (long long)K * ldm; if (n_ok > 0) gp[0] += tx; }
#if GRP
#define RG(K) { double *gp = Gcol + (long long)K * ldm; if (n_ok > 0) gp[0] = ga ? gp[0] + tx : tx; }
#else
#define RG(K) { if (n_ok > 0) Gcol[(long long)K * ldm] = tx; }
#endif
#endif

@TABLES@
extern "C" __global__ void __launch_bounds__(NT, 1) k_tree_gen(const TreeArgs a) {
  extern __shared__ __align__(16) char smraw[];
  double *val = (double *)smraw;
  double *adj = val + (size_t)a.n_val * A;
  double *esm = adj + (size_t)a.n_adj * A;
  const int al = threadIdx.x % AL, rl = threadIdx.x / AL;
  const char *vc = smraw + al * AR * 8;
  char *vw = smraw + al * AR * 8;
  char *ac = (char *)adj + al * AR * 8;
  const long long ldm = a.ldm;
  const unsigned ldm32 = (unsigned)a.ldm; (void)ldm32;
  const int n_groups = (a.c1 - a.c0 + A - 1) / A;
  for (int g = blockIdx.x; g < n_groups; g += gridDim.x) {
    const int atom0 = a.c0 + g * A + al * AR;
    const int n_ok = min(AR, max(0, a.c1 - atom0));
    const long long col = atom0 - a.c0;
    __syncthreads();
    for (int k = rl; k < a.n_basic; k += R)
      for (int r = 0; r < AR; ++r)
        val[(size_t)k * A + al * AR + r] = r < n_ok ? a.M[(long long)(GRP ? a.mload_k[k] : k) * ldm + col + r] : 0.0;
    if (a.want_adj)
      for (int k = rl; k < a.n_adj; k += R)
        for (int r = 0; r < AR; ++r) adj[(size_t)k * A + al * AR + r] = a.adj_init[k];
    if (GRP && a.want_adj && a.Sbar) {       // per-atom seeds of a group's cut nodes
      __syncthreads();
      for (int q = rl; q < a.n_cut; q += R)
        for (int r = 0; r < AR; ++r)
          adj[(size_t)a.cut_aslot[q] * A + al * AR + r] = r < n_ok ? a.Sbar[(long long)a.cut_row[q] * ldm + col + r] : 0.0;
    }
    __syncthreads();
    double ex = 0.0, ey = 0.0, ax = 0.0, ay = 0.0, tx = 0.0, ty = 0.0;
    (void)ey; (void)ay; (void)ty;
    {
      const char *s0 = vc;
@FWD@
    }
    {
      for (int q = rl; q < a.n_eseed; q += R) {
        const double sd = a.eseed_val[q];
        const double *v = val + (size_t)a.eseed_slot[q] * A + al * AR;
        ex = fma(sd, v[0], ex);
#if AR == 2
        ey = fma(sd, v[1], ey);
#endif
      }
      esm[rl * A + al * AR] = ex;
#if AR == 2
      esm[rl * A + al * AR + 1] = ey;
#endif
      if (a.B) {
        const int na = min(A, a.c1 - (a.c0 + g * A));
        for (int i = threadIdx.x; i < na * a.n_basis; i += NT) {
          const int at = i / a.n_basis, b = i - at * a.n_basis;
          a.B[(long long)(a.c0 + g * A + at) * a.n_basis + b] = val[(size_t)a.basis_slot[b] * A + at];
        }
      }
      __syncthreads();
      if (GRP && a.S)                          // cut values of a group, exported for the top program
        for (int q = rl; q < a.n_cut; q += R)
          for (int r = 0; r < AR; ++r)
            if (r < n_ok) a.S[(long long)a.cut_row[q] * ldm + col + r] = val[(size_t)a.cut_vslot[q] * A + al * AR + r];
      if (rl == 0 && a.write_energy) {
        for (int r = 0; r < AR; ++r) {
          if (r < n_ok) {
            double s = 0.0;
            for (int q = 0; q < R; ++q) s += esm[q * A + al * AR + r];
            const int z = (int)a.pos4[4 * (size_t)(atom0 + r) + 3];
            a.Ei[atom0 + r] = a.xi0[z] + s;
          }
        }
      }
    }
    if (!a.want_adj) continue;
    double *Gcol = a.G + col;
    const bool ga = a.g_accum != 0; (void)ga;
    for (int q = rl; q < a.n_gzero; q += R)
      for (int r = 0; r < AR; ++r)
        if (r < n_ok) Gcol[(long long)a.gzero_k[q] * ldm + r] = 0.0;
    {
      const char *s0 = ac;
@BWD@
    }
    __syncthreads();
    for (int q = rl; q < a.n_gseed; q += R)
      for (int r = 0; r < AR; ++r)
        if (r < n_ok) Gcol[(long long)a.gseed_k[q] * ldm + r] += a.gseed_val[q];
  }
}
)SRC";

void replace_all(std::string &s, const std::string &key, const std::string &val) {
  for (size_t p = s.find(key); p != std::string::npos; p = s.find(key, p + val.size())) s.replace(p, key.size(), val);
}

// straight-line source of one pass: per wave a switch over the row-lane, then the CTA barrier
// adj_init (backward pass of a whole table only): initial adjoints by slot, for the store-instead-of-add rows
// runs: when given, a run of >= kLineRun plain entries inside one group is emitted as a loop over a table of operand
// offsets (appended to *runs, emitted by the caller as the __device__ const array `l_off`) instead of 4 instructions
// per entry: the long backward groups are a quarter of the straight-line code, which is what bounds the kernel.
constexpr int kLineRun = 10;
constexpr size_t kMaxConstMul = 1024;      // doubles in the constant bank: 8 KB, what its cache holds (6000 cost 11 % at level 24)
static int line_run() { const char *e = getenv("MTP_TREE_RUN"); const int v = e ? atoi(e) : 0; return v >= 3 ? v : kLineRun; }
std::string gen_pass(const std::vector<TreeTerm> &prog, const std::vector<int32_t> &wave, int R, bool bwd,
                     const std::vector<double> &leaf_seed, int A, const std::vector<double> *adj_init = nullptr,
                     std::vector<unsigned> *runs = nullptr, std::vector<double> *cmul = nullptr) {
  std::string out;
  const int min_run = line_run();
  // multipliers and seeds: as operands from the constant bank (`cm[i]`, no instruction of their own) while the
  // bank has room, else as literals (two moves each)
  auto mref = [&](double v) {
    char t[40];
    if (cmul) {
      size_t i = 0;
      while (i < cmul->size() && memcmp(&(*cmul)[i], &v, 8) != 0) ++i;
      if (i == cmul->size() && cmul->size() < kMaxConstMul) cmul->push_back(v);
      if (i < cmul->size()) { snprintf(t, sizeof t, "cm[%zu]", i); return std::string(t); }
    }
    snprintf(t, sizeof t, "%a", v);
    return std::string(t);
  };
  std::vector<char> added(adj_init ? adj_init->size() : 0, 0);   // adjoint slots a row has already been added to
  out.reserve(prog.size() * 24);
  char buf[400];
  const unsigned row = (unsigned)A * 8u;
  for (size_t w = 0; w + 1 < wave.size(); ++w) {
    out += "      switch (rl) {\n";
    for (int l = 0; l < R; ++l) {
      int last = -1;
      for (int s = wave[w]; s < wave[w + 1]; ++s)
        if (prog[(size_t)s * R + l].a & kTreeRow) last = s;
      if (last < 0) continue;
      snprintf(buf, sizeof buf, "      case %d: {\n", l);
      out += buf;
      bool acc_open = false, tot_open = false;      // does acc / tot hold a partial sum?
      for (int s = wave[w]; s <= last; ++s) {
        int run = 0;                                  // plain entries from here to the end of the group
        if (runs && acc_open)
          for (int s2 = s; s2 <= last; ++s2) {
            const TreeTerm &q = prog[(size_t)s2 * R + l];
            if (bwd && (q.a & ~7u) == 0) break;
            ++run;
            if (q.a & kTreeGroup) break;
          }
        if (run >= min_run) {
          while (runs->size() & 3) runs->push_back(0);
          snprintf(buf, sizeof buf, "{const uint4*q=(const uint4*)(l_off+%zu);int n=%d;\n_Pragma(\"unroll 1\")\n"
                   "for(;n>=2;n-=2,++q){const uint4 v=LQ(q);E(v.x,v.y)E(v.z,v.w)}%s}",
                   runs->size(), run, (run & 1) ? "{const uint4 v=LQ(q);E(v.x,v.y)}" : "");
          out += buf;
          for (int s2 = s; s2 < s + run; ++s2) {
            const TreeTerm &q = prog[(size_t)s2 * R + l];
            runs->push_back(q.a & ~7u); runs->push_back(q.b & kTreeBMask);
          }
          s += run - 1;
        }
        const TreeTerm &t = prog[(size_t)s * R + l];
        if (run >= min_run) buf[0] = 0;
        else if (bwd && (t.a & ~7u) == 0) snprintf(buf, sizeof buf, "%s(%u)", acc_open ? "Y1" : "Y0", t.b & kTreeBMask);
        else snprintf(buf, sizeof buf, "%s(%u,%u)", acc_open ? "E" : "E0", t.a & ~7u, t.b & kTreeBMask);
        out += buf;
        acc_open = true;
        if (t.a & kTreeGroup) {
          if (!tot_open && t.mult == 1.0) snprintf(buf, sizeof buf, "G1()");
          else snprintf(buf, sizeof buf, "%s(%s)", tot_open ? "GC" : "G0", mref(t.mult).c_str());
          out += buf;
          acc_open = false; tot_open = true;
          if (t.a & kTreeRow) {
            const unsigned d = t.b >> kTreeDstShift;
            if (!bwd) {
              if (t.a & kTreeAlt) snprintf(buf, sizeof buf, "RL(%s)", mref(leaf_seed[d]).c_str());
              else snprintf(buf, sizeof buf, "RV(%u)", d * row);
            } else {
              if (t.a & kTreeAlt) snprintf(buf, sizeof buf, "RG(%u)", d);
              else if (t.b & kTreeAcc) snprintf(buf, sizeof buf, "RV(%u)", d * row);     // partial sum of a split row
              else if (adj_init && d < added.size() && !added[d]) {
                added[d] = 1;
                if ((*adj_init)[d] == 0.0) snprintf(buf, sizeof buf, "RS(%u)", d * row);
                else snprintf(buf, sizeof buf, "RI(%u,%s)", d * row, mref((*adj_init)[d]).c_str());
              }
              else snprintf(buf, sizeof buf, "RA(%u)", d * row);
            }
            out += buf;
            tot_open = false;
          }
        }
        out += "\n";
      }
      out += "      } break;\n";
    }
    out += "      default: break;\n      }\n      __syncthreads();\n";
  }
  return out;
}

// Shape-shared form of one pass (MTP_TREE_FORM=shared).  Rows of the same shape (entries per group, which
// multipliers are 1, how the row is disposed of) run ONE code body; what differs between them -- operand offsets,
// destination, multipliers, seeds -- comes from tables emitted as initialised __device__ const arrays and read
// through L1 (the constant bank was tried first: its cache is built for reuse, the tables are streamed).  A
// row-lane walks its rows of a wave in schedule order and dispatches on the shape, so every row does exactly the
// arithmetic of the straight-line form, in the same order (bit-identical), but the code is ~80 KB instead of
// ~220 KB at level 16 and stays in the instruction cache.
//   tables (prefix f / b): X_row[r] = {shape, first offset, first multiplier, 0}; X_beg[w * R + l] .. [w * R + l + 1] = rows of
//   row-lane l in wave w; X_off = byte offsets / destinations / run lengths, rows and runs padded to 16 bytes and
//   read four at a time; X_mul = multipliers, initial adjoints, leaf seeds.
// Returns the code; appends the tables to *tables and their size in bytes to *table_bytes.
constexpr int kRunLoop = 6;      // plain entries in a row of one group from which a run is looped
std::string gen_pass_shared(const std::vector<TreeTerm> &prog, const std::vector<int32_t> &wave, int R, bool bwd,
                            const std::vector<double> &leaf_seed, int A, const std::vector<double> *adj_init,
                            const char *pfx, std::string *tables, size_t *table_bytes) {
  std::vector<char> added(adj_init ? adj_init->size() : 0, 0);
  const unsigned row = (unsigned)A * 8u;
  std::vector<std::string> bodies;                 // code of shape i
  std::vector<std::string> keys;                   // its key
  std::vector<int> rows;                           // shape, off0, mul0 per row
  std::vector<int> beg;                            // [n_waves * R + 1]
  std::vector<unsigned> off;
  std::vector<double> mul;
  char buf[512];
  const size_t n_waves = wave.size() - 1;
  for (size_t w = 0; w < n_waves; ++w)
    for (int l = 0; l < R; ++l) {
      beg.push_back((int)rows.size() / 3);
      auto pad4 = [&] { while (off.size() & 3) off.push_back(0); };   // rows and runs start on 16 bytes: offsets are read four at a time
      pad4();
      int last = -1;
      for (int s = wave[w]; s < wave[w + 1]; ++s)
        if (prog[(size_t)s * R + l].a & kTreeRow) last = s;
      std::string key, body, seg;                 // seg: text of the current segment, whose offsets are loaded up front
      int seg_id = 0;
      auto tq = [&](int k) { char t[32]; snprintf(t, sizeof t, "a%d_%d.%c", seg_id, k >> 2, "xyzw"[k & 3]); return std::string(t); };
      int off0 = (int)off.size(), mul0 = (int)mul.size();
      bool acc_open = false, tot_open = false;
      int tcur = off0;                              // where the body's T4 points (moves past each run loop)
      auto close_seg = [&] {                        // declare the segment's offsets: one 16-byte constant load per four
        const int nq = ((int)off.size() - tcur + 3) / 4;
        for (int i = 0; i < nq; ++i) { char t[64]; snprintf(t, sizeof t, "const uint4 a%d_%d=LQ(T4+%d);", seg_id, i, i); body += t; }
        body += seg;
        seg.clear();
        ++seg_id;
      };
      for (int s = wave[w]; s <= last; ++s) {
        const int io = (int)off.size() - tcur;
        auto is_y = [&](const TreeTerm &q) { return bwd && (q.a & ~7u) == 0; };
        // a long run of plain entries inside one group becomes a loop with its length in the table, so that
        // rows which differ only in such lengths share a body (the FMA chain keeps its order)
        int run = 0;
        for (int s2 = s; s2 <= last; ++s2) {
          const TreeTerm &q = prog[(size_t)s2 * R + l];
          if (is_y(q)) break;
          ++run;
          if (q.a & kTreeGroup) break;
        }
        if (!acc_open) run = 0;                     // a group's first entry opens the accumulator outside the loop
        if (run >= kRunLoop) {
          off.push_back((unsigned)run);
          seg += "{int n=" + tq(io) + ";";
          pad4();
          const int qpos = ((int)off.size() - tcur) / 4;
          close_seg();
          snprintf(buf, sizeof buf, "const uint4*q=T4+%d;\n_Pragma(\"unroll 1\")\nfor(;n>=2;n-=2,++q){const uint4 v=LQ(q);E(v.x,v.y)E(v.z,v.w)}"
                   "if(n){const uint4 v=LQ(q);E(v.x,v.y)++q;}T4=q;}", qpos);
          body += buf;
          key += 'F';
          for (int s2 = s; s2 < s + run; ++s2) {
            const TreeTerm &q = prog[(size_t)s2 * R + l];
            off.push_back(q.a & ~7u); off.push_back(q.b & kTreeBMask);
          }
          pad4();
          tcur = (int)off.size();
          s += run - 1;
        }
        const TreeTerm &t = prog[(size_t)s * R + l];
        if (run >= kRunLoop) {
        } else if (is_y(t)) {
          seg += std::string(acc_open ? "Y1(" : "Y0(") + tq(io) + ")";
          off.push_back(t.b & kTreeBMask);
          key += 'y';
        } else {
          seg += std::string(acc_open ? "E(" : "E0(") + tq(io) + "," + tq(io + 1) + ")";
          off.push_back(t.a & ~7u); off.push_back(t.b & kTreeBMask);
          key += 'e';
        }
        acc_open = true;
        if (t.a & kTreeGroup) {
          if (!tot_open && t.mult == 1.0) { snprintf(buf, sizeof buf, "G1()"); key += '1'; }
          else {
            snprintf(buf, sizeof buf, "%s(__ldg(U+%d))", tot_open ? "GC" : "G0", (int)mul.size() - mul0);
            mul.push_back(t.mult);
            key += 'g';
          }
          seg += buf;
          acc_open = false; tot_open = true;
          if (t.a & kTreeRow) {
            const unsigned d = t.b >> kTreeDstShift;
            const int id = (int)off.size() - tcur, im = (int)mul.size() - mul0;
            if (!bwd) {
              if (t.a & kTreeAlt) { snprintf(buf, sizeof buf, "RL(__ldg(U+%d))", im); mul.push_back(leaf_seed[d]); key += 'L'; }
              else { snprintf(buf, sizeof buf, "RV(%s)", tq(id).c_str()); off.push_back(d * row); key += 'V'; }
            } else {
              if (t.a & kTreeAlt) { snprintf(buf, sizeof buf, "RG(%s)", tq(id).c_str()); off.push_back(d); key += 'G'; }
              else if (t.b & kTreeAcc) { snprintf(buf, sizeof buf, "RV(%s)", tq(id).c_str()); off.push_back(d * row); key += 'V'; }
              else if (adj_init && d < added.size() && !added[d]) {
                added[d] = 1;
                if ((*adj_init)[d] == 0.0) { snprintf(buf, sizeof buf, "RS(%s)", tq(id).c_str()); off.push_back(d * row); key += 'S'; }
                else { snprintf(buf, sizeof buf, "RI(%s,__ldg(U+%d))", tq(id).c_str(), im); off.push_back(d * row); mul.push_back((*adj_init)[d]); key += 'I'; }
              }
              else { snprintf(buf, sizeof buf, "RA(%s)", tq(id).c_str()); off.push_back(d * row); key += 'A'; }
            }
            seg += buf;
            close_seg();
            tot_open = false;
            seg_id = 0;
            // the row is complete: find or add its shape
            size_t sh = 0;
            while (sh < keys.size() && keys[sh] != key) ++sh;
            if (sh == keys.size()) { keys.push_back(key); bodies.push_back(body); }
            rows.push_back((int)sh); rows.push_back(off0); rows.push_back(mul0);
            key.clear(); body.clear();
            pad4();
            off0 = (int)off.size(); mul0 = (int)mul.size();
            tcur = off0;
          }
        }
      }
    }
  beg.push_back((int)rows.size() / 3);
  // ---- tables
  std::string &tb = *tables;
  const std::string P = pfx;
  tb += "__device__ const int4 " + P + "_row[] = {";
  for (size_t r = 0; r < rows.size() / 3; ++r) { snprintf(buf, sizeof buf, "{%d,%d,%d,0},", rows[3 * r], rows[3 * r + 1], rows[3 * r + 2]); tb += buf; }
  tb += "{0,0,0,0}};\n__device__ const int " + P + "_beg[] = {";
  for (int b : beg) { snprintf(buf, sizeof buf, "%d,", b); tb += buf; }
  tb += "0};\n__device__ const __align__(16) unsigned " + P + "_off[] = {";
  for (unsigned o : off) { snprintf(buf, sizeof buf, "%u,", o); tb += buf; }
  tb += "0};\n__device__ const double " + P + "_mul[] = {";
  for (double m : mul) { snprintf(buf, sizeof buf, "%a,", m); tb += buf; }
  tb += "0.0};\n";
  *table_bytes += rows.size() / 3 * 16 + 16 + beg.size() * 4 + 4 + off.size() * 4 + 4 + mul.size() * 8 + 8;
  // ---- code: one copy of every body per pass; the waves are a loop around the dispatch
  std::string out;
  snprintf(buf, sizeof buf, "      _Pragma(\"unroll 1\")\n      for (int w = 0; w < %zu; ++w) {\n", n_waves);
  out += buf;
  out += "      int r = __ldg(" + P + "_beg + w * R + rl); const int r1 = __ldg(" + P + "_beg + w * R + rl + 1);\n";
  out += "      int4 rn = __ldg(" + P + "_row + r);\n";
  out += "      for (; r < r1; ++r) {\n";
  // the row record is fetched one row ahead (the table ends with a spare record); prefetching the lines of the
  // other two streams a few rows ahead as well was measured and changed nothing
  out += "        const int4 rr = rn; rn = __ldg(" + P + "_row + r + 1);\n";
  out += "        const uint4 *T4 = (const uint4 *)(" + P + "_off + rr.y); const double *U = " + P + "_mul + rr.z;\n";
  out += "        switch (rr.x) {\n";
  for (size_t sh = 0; sh < keys.size(); ++sh) {
    snprintf(buf, sizeof buf, "        case %zu: { ", sh);
    out += buf;
    out += bodies[sh];
    out += " } break;\n";
  }
  out += "        default: break;\n        }\n      }\n      __syncthreads();\n      }\n";
  return out;
}
}  // namespace

// shared memory of the generated kernel: val + adj + energy partials [NT][AR]
size_t tree_jit_smem_bytes(int n_val, int n_adj, int AR, int NT) {
  return (((size_t)n_val + (size_t)n_adj) * 32 * AR * 8 + (size_t)NT * AR * 8 + 15) & ~(size_t)15;
}

struct TreeJit {
  cudaLibrary_t lib = nullptr;
  cudaKernel_t kernel = nullptr;
  int AR = 1, NT = 512;
};

void tree_jit_destroy(TreeJit *j) {
  if (!j) return;
  if (j->lib) cudaLibraryUnload(j->lib);
  delete j;
}

// Returns null (and a reason in *why) when the specialised kernel is not available.
// Host-only half: generate and compile the source of one schedule (thread-safe; mtp_create runs the
// programs of a partitioned table in parallel).  Empty result + reason when unavailable.
std::vector<char> tree_jit_compile(const TreeSched &sc, int AL, int AR, std::string *why) {
  std::vector<char> cubin;
  if (AL != 32) { *why = "codegen needs 32 atom-lanes"; return cubin; }
  const Nvrtc &rt = nvrtc();
  if (!rt.ok) { *why = "NVRTC not found"; return cubin; }
  const int R = sc.R, NT = R * AL;            // the schedule's row-lanes are this kernel's warps
  if (NT > 1024 || sc.A != AL * AR) { *why = "schedule shape mismatch"; return cubin; }
  std::string src = kFrame;
  replace_all(src, "@AR@", std::to_string(AR));
  replace_all(src, "@NT@", std::to_string(NT));
  replace_all(src, "@GRP@", sc.mload_k.empty() ? "0" : "1");
  // Two forms of the generated code: straight-line (default) and shape-shared bodies with operand tables
  // (MTP_TREE_FORM=shared; same arithmetic, bit-identical).  Measured at config 4: 2.82 ms against 4.08 ms -- the
  // shared form cures the instruction-fetch stall but pays for it in table-load latency and barrier imbalance
  // (DESIGN.md section 11), so it stays an option until that is fixed.
  std::string tables;
  size_t table_bytes = 0;
  const char *form = getenv("MTP_TREE_FORM");
  std::string fwd, bwd;
  if (form && form[0] == 's') {
    fwd = gen_pass_shared(sc.fprog, sc.fwave, R, false, sc.leaf_seed, AL * AR, nullptr, "f", &tables, &table_bytes);
    bwd = gen_pass_shared(sc.bprog, sc.bwave, R, true, sc.leaf_seed, AL * AR, sc.mload_k.empty() ? &sc.adj_init : nullptr, "b",
                          &tables, &table_bytes);
  }
  if (table_bytes == 0 || table_bytes > 60 * 1024) {      // larger tables: not measured, keep the straight-line form
    tables.clear();
    std::vector<unsigned> runs;                           // MTP_TREE_FORM=line: no run loops either (A/B measurements)
    // run loops for whole tables only: in the group programs of a partitioned table (level 24) they cost more in
    // serial latency than they save in fetch (tree 58.8 -> 61.2 ms even when limited to programs with few runs)
    std::vector<unsigned> *rp = ((form && form[0] == 'l') || (!sc.mload_k.empty() && !getenv("MTP_TREE_RUN"))) ? nullptr : &runs;
    std::vector<double> cmul;
    std::vector<double> *cp = (form && form[0] == 'l') ? nullptr : &cmul;
    fwd = gen_pass(sc.fprog, sc.fwave, R, false, sc.leaf_seed, AL * AR, nullptr, rp, cp);
    bwd = gen_pass(sc.bprog, sc.bwave, R, true, sc.leaf_seed, AL * AR, sc.mload_k.empty() ? &sc.adj_init : nullptr, rp, cp);
    // A loop iteration is a serial chain (table load -> address -> shared loads -> FMA): where most of a program
    // sits in long runs (the group programs of level 24: tree 58.8 -> 64.8 ms with loops) the loops themselves
    // become the critical path, so they are used only while the runs are a minority of the entries
    if (rp && !getenv("MTP_TREE_RUN") && (double)runs.size() / 2 > 0.4 * 3.0 * (double)sc.n_prod) {
      runs.clear(); cmul.clear();
      fwd = gen_pass(sc.fprog, sc.fwave, R, false, sc.leaf_seed, AL * AR, nullptr, nullptr, cp);
      bwd = gen_pass(sc.bprog, sc.bwave, R, true, sc.leaf_seed, AL * AR, sc.mload_k.empty() ? &sc.adj_init : nullptr, nullptr, cp);
    }
    if (!cmul.empty()) {
      tables += "__constant__ double cm[] = {";
      char t[40];
      for (double m : cmul) { snprintf(t, sizeof t, "%a,", m); tables += t; }
      tables += "0.0};\n";
    }
    if (!runs.empty()) {
      tables += "__device__ const __align__(16) unsigned l_off[] = {";
      char t[16];
      for (unsigned o : runs) { snprintf(t, sizeof t, "%u,", o); tables += t; }
      tables += "0,0,0,0};\n";
    }
  }
  replace_all(src, "@TABLES@", tables);
  replace_all(src, "@FWD@", fwd);
  replace_all(src, "@BWD@", bwd);
  if (const char *dump = getenv("MTP_TREE_DUMP")) {      // debugging aid: the generated source of the last compiled program
    if (FILE *f = fopen(dump, "w")) { fputs(src.c_str(), f); fclose(f); }
  }
  nvrtcProgram prog = nullptr;
  if (rt.CreateProgram(&prog, src.c_str(), "k_tree_gen.cu", 0, nullptr, nullptr) != 0) { *why = "nvrtcCreateProgram failed"; return cubin; }
  const char *opts[] = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo", "-default-device"};
  const int rc = rt.CompileProgram(prog, 4, opts);
  if (rc != 0) {
    size_t n = 0;
    std::string log;
    if (rt.GetProgramLogSize && rt.GetProgramLog && rt.GetProgramLogSize(prog, &n) == 0 && n > 1) { log.resize(n); rt.GetProgramLog(prog, &log[0]); }
    *why = "NVRTC compile failed: " + log.substr(0, 400);
    rt.DestroyProgram(&prog);
    return cubin;
  }
  size_t nbin = 0;
  rt.GetCUBINSize(prog, &nbin);
  cubin.resize(nbin);
  rt.GetCUBIN(prog, cubin.data());
  rt.DestroyProgram(&prog);
  return cubin;
}

// Device half: load a compiled schedule.
TreeJit *tree_jit_load(const std::vector<char> &cubin, int AR, int NT, std::string *why) {
  if (cubin.empty()) return nullptr;
  TreeJit *j = new TreeJit();
  j->AR = AR; j->NT = NT;
  cudaError_t e = cudaLibraryLoadData(&j->lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
  if (e == cudaSuccess) e = cudaLibraryGetKernel(&j->kernel, j->lib, "k_tree_gen");
  if (e == cudaSuccess) e = cudaFuncSetAttribute((const void *)j->kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 225 * 1024);
  if (e != cudaSuccess) {
    *why = std::string("loading the generated kernel failed: ") + cudaGetErrorString(e);
    cudaGetLastError();
    tree_jit_destroy(j);
    return nullptr;
  }
  return j;
}

TreeJit *tree_jit_build(const TreeSched &sc, int AL, int AR, std::string *why) {
  return tree_jit_load(tree_jit_compile(sc, AL, AR, why), AR, sc.R * AL, why);
}

cudaError_t tree_jit_launch(const TreeJit *j, const TreeArgs &a, cudaStream_t st) {
  const int Aat = 32 * j->AR;
  const int groups = (a.c1 - a.c0 + Aat - 1) / Aat;
  if (groups <= 0) return cudaSuccess;
  if (j->AR == 2 && ((a.ldm & 63) || ((uintptr_t)a.G & 15))) return cudaErrorMisalignedAddress;   // unpredicated G rows (RG)
  static int sms = 0;
  if (!sms) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev); }
  const size_t smem = tree_jit_smem_bytes(a.n_val, a.n_adj, j->AR, j->NT);
  int per_sm = (int)((227 * 1024) / (smem + 1024));
  per_sm = per_sm < 1 ? 1 : (per_sm > 2048 / j->NT ? 2048 / j->NT : per_sm);
  const int grid = groups < sms * per_sm ? groups : sms * per_sm;
  TreeArgs args = a;
  void *params[] = {&args};
  cudaError_t e = cudaLaunchKernel((const void *)j->kernel, dim3(grid), dim3(j->NT), params, smem, st);
  count_launch();
  return e;
}

}  // namespace mtpb
