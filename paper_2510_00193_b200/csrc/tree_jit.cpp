// K2 specialised at mtp_create time: the register program of tree_codegen.cpp (one atom per thread, node values
// and adjoints in a register window with Belady replacement, spills in private shared-memory columns) is put into
// a kernel frame, compiled with NVRTC for sm_100a and loaded through the runtime's library API.
// BASELINE.json north_star: "forward/adjoint contraction kernel with the tree in registers and shared memory".
//
// Memory layout the kernel relies on (kernels.h, kTile): every per-atom array of a chunk is tiled,
// [tile of 128 atoms][row][128], so a thread's element of row x sits at (its base pointer) + x * 1024 bytes --
// an immediate offset, no address arithmetic and no address registers.
//
// NVRTC is dlopen'ed.  Without it there is no specialised kernel: the caller records why (mtp_last_error) and
// the table interpreter of tree_kernel.cu runs instead -- both are CUDA paths.
#include <cuda_runtime.h>
#include <dlfcn.h>

#include <algorithm>
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
  std::string why;
};
const Nvrtc &nvrtc() {
  static Nvrtc n = [] {
    Nvrtc r;
    void *h = nullptr;
    for (const char *name : {"libnvrtc.so.12", "libnvrtc.so", "/usr/local/cuda/lib64/libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so"})
      if ((h = dlopen(name, RTLD_NOW | RTLD_LOCAL))) break;
    if (!h) { r.why = "libnvrtc.so.12 could not be loaded"; return r; }
    auto sym = [&](const char *s) { return dlsym(h, s); };
    r.CreateProgram = (decltype(r.CreateProgram))sym("nvrtcCreateProgram");
    r.CompileProgram = (decltype(r.CompileProgram))sym("nvrtcCompileProgram");
    r.GetCUBINSize = (decltype(r.GetCUBINSize))sym("nvrtcGetCUBINSize");
    r.GetCUBIN = (decltype(r.GetCUBIN))sym("nvrtcGetCUBIN");
    r.GetProgramLogSize = (decltype(r.GetProgramLogSize))sym("nvrtcGetProgramLogSize");
    r.GetProgramLog = (decltype(r.GetProgramLog))sym("nvrtcGetProgramLog");
    r.DestroyProgram = (decltype(r.DestroyProgram))sym("nvrtcDestroyProgram");
    r.ok = r.CreateProgram && r.CompileProgram && r.GetCUBINSize && r.GetCUBIN && r.DestroyProgram;
    if (!r.ok) r.why = "libnvrtc lacks the expected entry points";
    return r;
  }();
  return n;
}

// Kernel frame; @PRE@ = constant table and K2_SLOTS / K2_ENERGY, @BODY@ = the register program.
// Loads of spilled values are opaque to the compiler (asm volatile), so that it neither forwards a spilled value
// through a register nor merges the reload of an evicted input with its first load: the register budget is the
// generator's.  First loads of the inputs are plain non-coherent loads the scheduler may hoist.
const char *kFrame = R"SRC(
typedef unsigned long long size_t_;
struct K2Args {
  const double *in; double *out; const double *sbar; double *sout; double *bt; double *Ei;
  const double *xi0; const double *pos4;
  int n_io, n_cut, n_bt, c0, n;
  const double *cmx;
};
@PRE@
#define T @T@
template <int OFF> __device__ __forceinline__ double ldnc(const double *p) { double v; asm("ld.global.nc.f64 %0, [%1+%2];" : "=d"(v) : "l"(p), "n"(OFF)); return v; }
template <int OFF> __device__ __forceinline__ double ldvol(const double *p) { double v; asm volatile("ld.volatile.global.f64 %0, [%1+%2];" : "=d"(v) : "l"(p), "n"(OFF)); return v; }
template <int OFF> __device__ __forceinline__ double ldgl(const double *p) { double v; asm volatile("ld.global.f64 %0, [%1+%2];" : "=d"(v) : "l"(p), "n"(OFF)); return v; }
template <int OFF> __device__ __forceinline__ void stgl(double *p, double v) { asm volatile("st.global.f64 [%0+%1], %2;" :: "l"(p), "n"(OFF), "d"(v)); }
template <int OFF> __device__ __forceinline__ double lds(unsigned a) { double v; asm volatile("ld.shared.f64 %0, [%1+%2];" : "=d"(v) : "r"(a), "n"(OFF)); return v; }
template <int OFF> __device__ __forceinline__ void sts(unsigned a, double v) { asm volatile("st.shared.f64 [%0+%1], %2;" :: "r"(a), "n"(OFF), "d"(v)); }
#define PFALL() asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(IN), "r"(a.n_io * 1024) : "memory")
#define LI(x) ldnc<(x) * 1024>(IN)
#define LR(x) ldvol<(x) * 1024>(IN)
#define LB(x) ldnc<(x) * 1024>(SBAR)
#define LO(x) ldgl<(x) * 1024>(OUT)
#define SO(x, v) stgl<(x) * 1024>(OUT, v)
#define LS(x) lds<(x) * (T * 8)>(sma)
#define SS(x, v) sts<(x) * (T * 8)>(sma, v)
#define SC(x, v) stgl<(x) * 1024>(SOUT, v)
#define SB(x, v) stgl<(x) * 1024>(BT, v)
extern "C" __global__ void __launch_bounds__(T, @MINB@) k2(const K2Args a) {
  extern __shared__ double sm[];
  const int col = blockIdx.x * T + threadIdx.x;
  if (col >= a.n) return;
  const unsigned sma = (unsigned)__cvta_generic_to_shared(sm + threadIdx.x); (void)sma;
  const size_t_ tile = (size_t_)(col >> 7) * 128, lane = col & 127;
  const double *IN = a.in + tile * a.n_io + lane; (void)IN;
  double *OUT = a.out + tile * a.n_io + lane; (void)OUT;
  const double *SBAR = a.sbar + tile * a.n_cut + lane; (void)SBAR;
  double *SOUT = a.sout + tile * a.n_cut + lane; (void)SOUT;
  double *BT = a.bt + tile * a.n_bt + lane; (void)BT;
  // Whoever starts a tile asks L2 for what the tile's threads will read row by row over their whole run
  // (K2_PREFETCH: one bulk prefetch of the input block): without it every first touch of a row pays the HBM
  // latency with only 8 warps per SM to hide it
  if (lane == 0) { K2_PREFETCH }
  double e = 0.0; (void)e;
@BODY@
#if K2_ENERGY
  { const int at = a.c0 + col; const int z = (int)a.pos4[4 * (size_t_)at + 3]; a.Ei[at] = a.xi0[z] + e; }
#endif
}
)SRC";

void replace_all(std::string &s, const std::string &key, const std::string &val) {
  for (size_t p = s.find(key); p != std::string::npos; p = s.find(key, p + val.size())) s.replace(p, key.size(), val);
}
}  // namespace

bool k2_jit_available(std::string *why) {
  const Nvrtc &rt = nvrtc();
  if (!rt.ok && why) *why = rt.why;
  return rt.ok;
}

// threads per CTA and CTAs per SM for a program with this many shared-memory slots per thread: as many threads per
// SM as the slots allow (227 KB per SM), in CTAs of at most 128 threads
void k2_shape(int n_slots, int *threads, int *ctas_per_sm) {
  const size_t cap = 227 * 1024 - 2048;
  const size_t per_thread = (size_t)(n_slots > 0 ? n_slots : 1) * 8;
  *threads = 128; *ctas_per_sm = 2;
  if (per_thread * 128 * 2 + 2 * 1024 <= cap) return;
  *ctas_per_sm = 1;
  for (int t = 128; t >= 32; t >>= 1) { *threads = t; if (per_thread * t <= cap) return; }
  *threads = 0;                             // does not fit at all
}

std::string k2_source(const K2Gen &g) {
  int threads = 0, minb = 1;
  k2_shape(g.n_slots, &threads, &minb);
  std::string src = kFrame;
  replace_all(src, "@T@", std::to_string(threads));
  replace_all(src, "@MINB@", std::to_string(minb));
  replace_all(src, "@PRE@", g.source);
  replace_all(src, "@BODY@", g.body);
  return src;
}

// Host-only half (thread-safe): compile one generated program.  Empty result + reason when unavailable.
std::vector<char> k2_jit_compile(const K2Gen &g, std::string *why) {
  std::vector<char> cubin;
  const Nvrtc &rt = nvrtc();
  if (!rt.ok) { *why = rt.why; return cubin; }
  int threads = 0, minb = 1;
  k2_shape(g.n_slots, &threads, &minb);
  if (threads == 0) { *why = "register program needs more shared memory than an SM has"; return cubin; }
  const std::string src = k2_source(g);
  nvrtcProgram prog = nullptr;
  if (rt.CreateProgram(&prog, src.c_str(), "k2.cu", 0, nullptr, nullptr) != 0) { *why = "nvrtcCreateProgram failed"; return cubin; }
  const char *opts[] = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo"};
  const int rc = rt.CompileProgram(prog, 3, opts);
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

struct K2Kernel {
  cudaLibrary_t lib = nullptr;
  cudaKernel_t kernel = nullptr;
  int threads = 128;
  size_t smem = 0;
  double *cmx = nullptr;        // constants beyond the constant bank
};

void k2_jit_destroy(K2Kernel *k) {
  if (!k) return;
  if (k->lib) cudaLibraryUnload(k->lib);
  if (k->cmx) cudaFree(k->cmx);
  delete k;
}

// Device half: load a compiled program.
K2Kernel *k2_jit_load(const std::vector<char> &cubin, int n_slots, const std::vector<double> &consts, std::string *why) {
  if (cubin.empty()) return nullptr;
  K2Kernel *k = new K2Kernel();
  int minb = 1;
  k2_shape(n_slots, &k->threads, &minb);
  k->smem = (size_t)n_slots * 8 * k->threads;
  cudaError_t e = cudaLibraryLoadData(&k->lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
  if (e == cudaSuccess) e = cudaLibraryGetKernel(&k->kernel, k->lib, "k2");
  if (e == cudaSuccess && k->smem > 48 * 1024)
    e = cudaFuncSetAttribute((const void *)k->kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k->smem);
  if (e == cudaSuccess && !consts.empty()) {           // the weights-dependent constants: bank first, overflow in global memory
    void *cm = nullptr;
    size_t bytes = 0;
    e = cudaLibraryGetGlobal(&cm, &bytes, k->lib, "cm");
    const size_t nbank = std::min(consts.size(), (size_t)kK2ConstBank);
    if (e == cudaSuccess && bytes < nbank * 8) e = cudaErrorInvalidValue;
    if (e == cudaSuccess) e = cudaMemcpy(cm, consts.data(), nbank * 8, cudaMemcpyHostToDevice);
    if (e == cudaSuccess && consts.size() > (size_t)kK2ConstBank) {
      e = cudaMalloc((void **)&k->cmx, consts.size() * 8);
      if (e == cudaSuccess) e = cudaMemcpy(k->cmx, consts.data(), consts.size() * 8, cudaMemcpyHostToDevice);
    }
  }
  if (e != cudaSuccess) {
    *why = std::string("loading the generated kernel failed: ") + cudaGetErrorString(e);
    cudaGetLastError();
    k2_jit_destroy(k);
    return nullptr;
  }
  return k;
}

cudaError_t k2_jit_launch(const K2Kernel *k, const K2Args &a, cudaStream_t st) {
  if (a.n <= 0) return cudaSuccess;
  const int grid = (a.n + k->threads - 1) / k->threads;
  K2Args args = a;
  args.cmx = k->cmx;
  void *params[] = {&args};
  cudaError_t e = cudaLaunchKernel((const void *)k->kernel, dim3(grid), dim3(k->threads), params, k->smem, st);
  count_launch();
  return e;
}

}  // namespace mtpb
