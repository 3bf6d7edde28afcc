// K2: forward contraction tree (a5: B_alpha, E_i) and its adjoint sweep (a6: G = dE_i/dM).
// BASELINE.json north_star: "forward/adjoint contraction kernel with the tree in registers and
// shared memory".  A CTA of 128 threads owns AL atoms; node values and adjoints of those atoms
// live in shared memory as [node][AL]; thread (rl, al) walks the items rl, rl+R, ... of each
// wave for atom al (R = 128/AL row-lanes).  The table is read once per CTA per wave through
// L1/L2 (identical for all atoms).
#include <cuda_runtime.h>

#include "kernels.h"

namespace mtpb {

template <int AL>
__global__ void __launch_bounds__(128) k_tree(const TreeArgs a) {
  extern __shared__ double sm[];
  constexpr int R = 128 / AL;
  double *val = sm;
  double *adj = sm + (size_t)a.n_nodes * AL;
  const int al = threadIdx.x % AL, rl = threadIdx.x / AL;
  const int atom = a.c0 + blockIdx.x * AL + al;
  const bool act = atom < a.c1;
  const long long col = atom - a.c0;
  for (int k = rl; k < a.n_nodes; k += R) {
    double v = 0.0;
    if (k < a.n_basic && act) v = a.M[(long long)k * a.ldm + col];
    val[k * AL + al] = v;
    adj[k * AL + al] = 0.0;
  }
  __syncthreads();
  // ---- forward
  for (int w = 0; w < a.nfw; ++w) {
    const int lo = a.fwave[w], hi = a.fwave[w + 1];
    for (int it = lo + rl; it < hi; it += R) {
      const int4 I = __ldg(reinterpret_cast<const int4 *>(a.fitems) + it);
      if (I.z <= 0) continue;
      const int4 *tp = reinterpret_cast<const int4 *>(a.fterms) + I.y;
      double acc = 0.0;
#pragma unroll 4
      for (int k = 0; k < I.z; ++k) {
        const int4 T = __ldg(tp + k);
        const double m = __hiloint2double(T.w, T.z);
        const int na = T.x & 0xffff, nb = (unsigned)T.x >> 16;
        acc = fma(m * val[na * AL + al], val[nb * AL + al], acc);
      }
      val[I.x * AL + al] = acc;
    }
    __syncthreads();
  }
  // ---- energy, basis values, adjoint seeds
  {
    double e = 0.0;
    for (int b = rl; b < a.n_basis; b += R) {
      const int n = a.basis_node[b];
      const double v = val[n * AL + al], x = a.xi[b];
      e = fma(x, v, e);
      if (a.B && act) a.B[(long long)atom * a.n_basis + b] = v;
    }
    // reduce e over the R row-lanes of this atom through shared memory, fixed order
    __shared__ double esm[128];
    esm[threadIdx.x] = e;
    __syncthreads();
    if (rl == 0 && act) {
      double s = 0.0;
      for (int r = 0; r < R; ++r) s += esm[r * AL + al];
      const int z = (int)a.pos4[4 * (size_t)atom + 3];
      a.Ei[atom] = a.xi0[z] + s;
    }
  }
  if (!a.want_adj) return;
  for (int q = rl; q < a.n_seed; q += R) adj[a.seed_node[q] * AL + al] = a.seed_val[q];
  __syncthreads();
  // ---- backward
  for (int w = 0; w < a.nbw; ++w) {
    const int lo = a.bwave[w], hi = a.bwave[w + 1];
    for (int it = lo + rl; it < hi; it += R) {
      const int4 I = __ldg(reinterpret_cast<const int4 *>(a.bitems) + it);
      if (I.z <= 0) continue;
      const int4 *tp = reinterpret_cast<const int4 *>(a.bterms) + I.y;
      double acc = 0.0;
#pragma unroll 4
      for (int k = 0; k < I.z; ++k) {
        const int4 T = __ldg(tp + k);
        const double m = __hiloint2double(T.w, T.z);
        const int nd = T.x & 0xffff, no = (unsigned)T.x >> 16;
        acc = fma(m * adj[nd * AL + al], val[no * AL + al], acc);
      }
      adj[I.x * AL + al] += acc;
    }
    __syncthreads();
  }
  if (act)
    for (int k = rl; k < a.n_basic; k += R) a.G[(long long)k * a.ldm + col] = adj[k * AL + al];
}

size_t tree_smem_bytes(int n_nodes, int AL) { return (size_t)n_nodes * AL * 16; }

int tree_pick_al(int n_nodes) {
  // largest AL <= 16 that lets two CTAs share an SM, else the largest that fits at all
  for (int al = 16; al >= 1; al >>= 1)
    if (tree_smem_bytes(n_nodes, al) <= 100 * 1024) return al;
  for (int al = 16; al >= 1; al >>= 1)
    if (tree_smem_bytes(n_nodes, al) <= 220 * 1024) return al;
  return 0;
}

template <int AL>
static cudaError_t launch_al(const TreeArgs &a, cudaStream_t st) {
  const size_t smem = tree_smem_bytes(a.n_nodes, AL);
  static bool attr_done = false;
  if (!attr_done) {
    cudaError_t e = cudaFuncSetAttribute(k_tree<AL>, cudaFuncAttributeMaxDynamicSharedMemorySize, 225 * 1024);
    if (e != cudaSuccess) return e;
    attr_done = true;
  }
  const int n = a.c1 - a.c0;
  const int grid = (n + AL - 1) / AL;
  if (grid <= 0) return cudaSuccess;
  k_tree<AL><<<grid, 128, smem, st>>>(a);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_tree(const TreeArgs &a, int AL, cudaStream_t st) {
  switch (AL) {
    case 1: return launch_al<1>(a, st);
    case 2: return launch_al<2>(a, st);
    case 4: return launch_al<4>(a, st);
    case 8: return launch_al<8>(a, st);
    case 16: return launch_al<16>(a, st);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace mtpb
