// K2: forward contraction tree (a5: B_alpha, E_i) and its adjoint sweep (a6: G = dE_i/dM).
// BASELINE.json north_star: "forward/adjoint contraction kernel with the tree in registers and
// shared memory".  A CTA of 128 threads owns AL atoms; node values and adjoints of those atoms
// live in shared memory as [node][AL]; thread (rl, al) walks the items rl, rl+R, ... of each
// wave for its AR atoms (R = 128/AL row-lanes, A = AL*AR atoms per CTA).  The table is read once per CTA per wave through
// L1/L2 (identical for all atoms).
#include <cuda_runtime.h>

#include "kernels.h"

namespace mtpb {

// row stride (doubles) of the [node][atom] arrays: +2 spreads rows of different nodes over the banks
__host__ __device__ constexpr int tree_ld(int A) { return A >= 4 ? A + 2 : A; }

template <int AR>
__device__ __forceinline__ void ldv(const double *p, double (&v)[AR]) {
  if (AR == 1) { v[0] = p[0]; }
  else {
#pragma unroll
    for (int j = 0; j < AR; j += 2) { const double2 t = *reinterpret_cast<const double2 *>(p + j); v[j] = t.x; v[j + 1] = t.y; }
  }
}
template <int AR>
__device__ __forceinline__ void stv(double *p, const double (&v)[AR]) {
  if (AR == 1) { p[0] = v[0]; }
  else {
#pragma unroll
    for (int j = 0; j < AR; j += 2) *reinterpret_cast<double2 *>(p + j) = make_double2(v[j], v[j + 1]);
  }
}

// One wave of the lane-major program (tree.h): thread (rl, al) executes entry [s][rl] of every
// step s for its AR atoms (register blocking: one table read and one decode serve AR atoms).
// Entries are prefetched kTreePrefetch steps ahead; a warp's reads of one step are contiguous.
template <int LD, int AR, int R, bool BWD>
__device__ __forceinline__ void run_wave(const TreeTerm *__restrict__ prog, int lo, int hi, int rl,
                                         const double *__restrict__ val, double *adj, double *valw, int cb) {
  constexpr int PF = kTreePrefetch;
  const double *src0 = BWD ? adj : val;
  const int4 *p = reinterpret_cast<const int4 *>(prog) + (size_t)lo * R + rl;
  int4 T[PF];
#pragma unroll
  for (int u = 0; u < PF; ++u) T[u] = __ldg(p + (size_t)u * R);
  double acc[AR];
#pragma unroll
  for (int r = 0; r < AR; ++r) acc[r] = 0.0;
  for (int s = lo; s < hi; s += PF) {
    p += (size_t)PF * R;
#pragma unroll
    for (int u = 0; u < PF; ++u) {
      const int4 t = T[u];
      T[u] = __ldg(p + (size_t)u * R);          // padded past the end of the program
      const double m = __hiloint2double(t.w, t.z);
      const int na = t.x & 0xffff, nb = (unsigned)t.x >> 16;
      double x[AR], y[AR];
      ldv<AR>(src0 + na * LD + cb, x);
      ldv<AR>(val + nb * LD + cb, y);
#pragma unroll
      for (int r = 0; r < AR; ++r) acc[r] = fma(m * x[r], y[r], acc[r]);
      if ((unsigned)t.y >> 16) {                 // entry closes a row
        double *dst = (BWD ? adj : valw) + (t.y & 0xffff) * LD + cb;
        if (BWD) {
          double old[AR];
          ldv<AR>(dst, old);
#pragma unroll
          for (int r = 0; r < AR; ++r) acc[r] += old[r];
        }
        stv<AR>(dst, acc);
#pragma unroll
        for (int r = 0; r < AR; ++r) acc[r] = 0.0;
      }
    }
  }
}

template <int AL, int AR>
__global__ void __launch_bounds__(128) k_tree(const TreeArgs a) {
  extern __shared__ __align__(16) double sm[];
  constexpr int A = AL * AR, R = 128 / AL, LD = tree_ld(A);
  double *val = sm;
  double *adj = sm + (size_t)a.n_nodes * LD;
  const int al = threadIdx.x % AL, rl = threadIdx.x / AL, cb = al * AR;
  const int atom0 = a.c0 + blockIdx.x * A + cb;       // this thread's first atom
  const long long col0 = atom0 - a.c0;
  for (int k = rl; k < a.n_nodes; k += R) {
    double v[AR], z[AR];
#pragma unroll
    for (int r = 0; r < AR; ++r) {
      v[r] = (k < a.n_basic && atom0 + r < a.c1) ? a.M[(long long)k * a.ldm + col0 + r] : 0.0;
      z[r] = 0.0;
    }
    stv<AR>(val + k * LD + cb, v);
    stv<AR>(adj + k * LD + cb, z);
  }
  __syncthreads();
  for (int w = 0; w < a.nfw; ++w) {
    run_wave<LD, AR, R, false>(a.fprog, a.fwave[w], a.fwave[w + 1], rl, val, adj, val, cb);
    __syncthreads();
  }
  // ---- energy and basis values
  {
    double e[AR];
#pragma unroll
    for (int r = 0; r < AR; ++r) e[r] = 0.0;
    for (int b = rl; b < a.n_basis; b += R) {
      const int n = a.basis_node[b];
      const double x = a.xi[b];
      double v[AR];
      ldv<AR>(val + n * LD + cb, v);
#pragma unroll
      for (int r = 0; r < AR; ++r) {
        e[r] = fma(x, v[r], e[r]);
        if (a.B && atom0 + r < a.c1) a.B[(long long)(atom0 + r) * a.n_basis + b] = v[r];
      }
    }
    __shared__ double esm[128 * AR];       // fixed-order reduction over the R row-lanes
#pragma unroll
    for (int r = 0; r < AR; ++r) esm[threadIdx.x * AR + r] = e[r];
    __syncthreads();
    if (rl == 0) {
#pragma unroll
      for (int r = 0; r < AR; ++r) {
        if (atom0 + r < a.c1) {
          double s = 0.0;
          for (int q = 0; q < R; ++q) s += esm[(q * AL + al) * AR + r];
          const int z = (int)a.pos4[4 * (size_t)(atom0 + r) + 3];
          a.Ei[atom0 + r] = a.xi0[z] + s;
        }
      }
    }
  }
  if (!a.want_adj) return;
  for (int q = rl; q < a.n_seed; q += R) {
    double v[AR];
#pragma unroll
    for (int r = 0; r < AR; ++r) v[r] = a.seed_val[q];
    stv<AR>(adj + a.seed_node[q] * LD + cb, v);
  }
  __syncthreads();
  for (int w = 0; w < a.nbw; ++w) {
    run_wave<LD, AR, R, true>(a.bprog, a.bwave[w], a.bwave[w + 1], rl, val, adj, val, cb);
    __syncthreads();
  }
  for (int k = rl; k < a.n_basic; k += R) {
    double g[AR];
    ldv<AR>(adj + k * LD + cb, g);
#pragma unroll
    for (int r = 0; r < AR; ++r)
      if (atom0 + r < a.c1) a.G[(long long)k * a.ldm + col0 + r] = g[r];
  }
}

size_t tree_smem_bytes(int n_nodes, int A) { return (size_t)n_nodes * tree_ld(A) * 16; }

int tree_pick_al(int n_nodes) {
  // largest AL <= 16 that lets two CTAs share an SM, else the largest that fits at all
  for (int al = 16; al >= 1; al >>= 1)
    if (tree_smem_bytes(n_nodes, al) <= 100 * 1024) return al;
  for (int al = 16; al >= 1; al >>= 1)
    if (tree_smem_bytes(n_nodes, al) <= 220 * 1024) return al;
  return 0;
}

template <int AL, int AR>
static cudaError_t launch_al(const TreeArgs &a, cudaStream_t st) {
  constexpr int A = AL * AR;
  const size_t smem = tree_smem_bytes(a.n_nodes, A);
  static bool attr_done = false;
  if (!attr_done) {
    cudaError_t e = cudaFuncSetAttribute(k_tree<AL, AR>, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024);
    if (e != cudaSuccess) return e;
    attr_done = true;
  }
  const int n = a.c1 - a.c0;
  const int grid = (n + A - 1) / A;
  if (grid <= 0) return cudaSuccess;
  k_tree<AL, AR><<<grid, 128, smem, st>>>(a);
  count_launch();
  return cudaGetLastError();
}

// A = atoms per CTA; AR = min(4, A) atoms per thread, AL = A / AR atom-lanes, R = 128 / AL row-lanes
int tree_row_lanes(int A) { const int AR = A < 4 ? A : 4; return 128 / (A / AR); }

cudaError_t launch_tree(const TreeArgs &a, int A, cudaStream_t st) {
  switch (A) {
    case 1: return launch_al<1, 1>(a, st);
    case 2: return launch_al<1, 2>(a, st);
    case 4: return launch_al<1, 4>(a, st);
    case 8: return launch_al<2, 4>(a, st);
    case 16: return launch_al<4, 4>(a, st);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace mtpb
