// K2: forward contraction tree (a5: B_alpha, E_i) and its adjoint sweep (a6: G = dE_i/dM).
// BASELINE.json north_star: "forward/adjoint contraction kernel with the tree in registers and
// shared memory".  Persistent CTAs loop over groups of A = AL*AR atoms.  Thread (rl, al) owns
// the AR atoms of atom-lane al and is row-lane rl of R = NT/AL; node values val[slot][A] and
// the adjoints of the intermediate nodes adj[slot][A] live in shared memory (tree.h explains
// which nodes get a slot).  Row-lane rl executes entry [s][rl] of every step s of the
// lane-major program.  With AL = 32 a warp is one row-lane: the 16-byte entry is warp-uniform,
// every shared access is a conflict-free full row, M is read and G written as full lines; AR = 2
// halves the decode work per atom.  The adjoints of the packed moments (the last backward
// wave) go straight to global memory.  The program is staged in shared memory once per CTA when
// it fits, else streamed through L1/L2 (it is identical for all CTAs).
#include <cuda_runtime.h>

#include "kernels.h"

namespace mtpb {

template <int AR>
struct Vec { double v[AR]; };
template <int AR>
__device__ __forceinline__ Vec<AR> lds(const char *p) {
  Vec<AR> r;
  if (AR == 1) r.v[0] = *reinterpret_cast<const double *>(p);
  else { const double2 t = *reinterpret_cast<const double2 *>(p); r.v[0] = t.x; r.v[AR - 1] = t.y; }
  return r;
}
template <int AR>
__device__ __forceinline__ void sts(char *p, const Vec<AR> &x) {
  if (AR == 1) *reinterpret_cast<double *>(p) = x.v[0];
  else *reinterpret_cast<double2 *>(p) = make_double2(x.v[0], x.v[AR - 1]);
}

// One pass (all forward waves, or all backward waves) of the lane-major program.  The entries of a
// row-lane form one contiguous strided stream across the waves, so a PF-deep register queue of
// entries is kept full over the whole pass (from the shared-memory copy of the program when PS,
// else through L1/L2); waves end on multiples of kTreePrefetch steps, where the CTA barrier sits.
//   fwd: acc += val[a] * val[b];        bwd: acc += adj[a] * val[b]
//   group close: tot += mult * acc;     row close: store / accumulate tot (tree.h kTreeAlt)
template <int AL, int AR, int R, bool BWD, bool PS>
__device__ __forceinline__ void run_pass(const int4 *__restrict__ prog, const int *__restrict__ wave, int n_waves,
                                         int rl, const char *__restrict__ val, char *adj, char *valw,
                                         const double *__restrict__ leaf_seed, Vec<AR> &e,
                                         double *__restrict__ Gcol, int n_ok, bool g_accum) {
  constexpr int BL = kTreePrefetch;            // block: entries between two wave-boundary checks
  constexpr int NB = PS ? 1 : 4;               // blocks in the queue: 4 entries ahead from shared memory, 16 from L2
  constexpr int PF = BL * NB;
  constexpr unsigned ROW = AL * AR * 8;
  if (n_waves <= 0) return;
  const char *src0 = BWD ? adj : val;
  const int4 *p = prog + rl;                   // entry of step 0
  int4 T[PF];
#pragma unroll
  for (int u = 0; u < PF; ++u) T[u] = PS ? p[(size_t)u * R] : __ldg(p + (size_t)u * R);
  Vec<AR> acc, tot;
#pragma unroll
  for (int r = 0; r < AR; ++r) { acc.v[r] = 0.0; tot.v[r] = 0.0; }
  int s = 0, w = 0, hi = wave[1];
  while (true) {
#pragma unroll
    for (int q = 0; q < NB; ++q) {
      while (s >= hi) {                        // wave boundary (uniform over the CTA)
        __syncthreads();
        if (++w == n_waves) return;
        hi = wave[w + 1];
#pragma unroll
        for (int r = 0; r < AR; ++r) { acc.v[r] = 0.0; tot.v[r] = 0.0; }   // drop what the no-op padding added
      }
#pragma unroll
      for (int v = 0; v < BL; ++v) {
        const int u = q * BL + v;
        const int4 t = T[u];
        const Vec<AR> x = lds<AR>(src0 + ((unsigned)t.x & ~7u));
        const Vec<AR> y = lds<AR>(val + ((unsigned)t.y & kTreeBMask));
#pragma unroll
        for (int r = 0; r < AR; ++r) acc.v[r] = fma(x.v[r], y.v[r], acc.v[r]);
        if (t.x & (int)kTreeGroup) {
          const double m = __hiloint2double(t.w, t.z);
#pragma unroll
          for (int r = 0; r < AR; ++r) { tot.v[r] = fma(m, acc.v[r], tot.v[r]); acc.v[r] = 0.0; }
          if (t.x & (int)kTreeRow) {
            const unsigned d = (unsigned)t.y >> kTreeDstShift;
            if (!BWD) {
              if (t.x & (int)kTreeAlt) {
                const double sd = __ldg(leaf_seed + d);
#pragma unroll
                for (int r = 0; r < AR; ++r) e.v[r] = fma(sd, tot.v[r], e.v[r]);
              } else {
                sts<AR>(valw + d * ROW, tot);
              }
            } else if (t.x & (int)kTreeAlt) {
#pragma unroll
              for (int r = 0; r < AR; ++r)
                if (r < n_ok) {
                  double *gp = Gcol + d * kTile + r;
                  *gp = g_accum ? *gp + tot.v[r] : tot.v[r];
                }
            } else if (t.y & (int)kTreeAcc) {          // piece of a split row: partial sum into a spare val slot
              sts<AR>(valw + d * ROW, tot);
            } else {
              char *qd = adj + d * ROW;               // adj was initialised with the node's seed
              Vec<AR> old = lds<AR>(qd);
#pragma unroll
              for (int r = 0; r < AR; ++r) old.v[r] += tot.v[r];
              sts<AR>(qd, old);
            }
#pragma unroll
            for (int r = 0; r < AR; ++r) tot.v[r] = 0.0;
          }
        }
        // refill the slot PF steps ahead (the program is padded past its end)
        T[u] = PS ? p[(size_t)(s + v + PF) * R] : __ldg(p + (size_t)(s + v + PF) * R);
      }
      s += BL;
    }
  }
}

template <int AL, int AR, int NT, bool PS>
__global__ void __launch_bounds__(NT) k_tree(const TreeArgs a) {
  extern __shared__ __align__(16) char smraw[];
  constexpr int R = NT / AL, A = AL * AR;
  double *val = reinterpret_cast<double *>(smraw);
  double *adj = val + (size_t)a.n_val * A;
  double *esm = adj + (size_t)a.n_adj * A;            // [NT][AR] energy partials
  int *wsm = reinterpret_cast<int *>(esm + NT * AR);  // wave offsets: fwave [nfw+1], bwave [nbw+1]
  const int4 *fprog = reinterpret_cast<const int4 *>(a.fprog), *bprog = reinterpret_cast<const int4 *>(a.bprog);
  for (int i = threadIdx.x; i <= a.nfw; i += NT) wsm[i] = a.fwave[i];
  for (int i = threadIdx.x; i <= a.nbw; i += NT) wsm[a.nfw + 1 + i] = a.bwave[i];
  if (PS) {
    int4 *psm = reinterpret_cast<int4 *>(smraw + a.prog_smem_off);
    for (int i = threadIdx.x; i < a.n_fprog; i += NT) psm[i] = __ldg(fprog + i);
    for (int i = threadIdx.x; i < a.n_bprog; i += NT) psm[a.n_fprog + i] = __ldg(bprog + i);
    fprog = psm; bprog = psm + a.n_fprog;
  }
  const int *fw = wsm, *bw = wsm + a.nfw + 1;
  const int al = threadIdx.x % AL, rl = threadIdx.x / AL;
  const char *valc = smraw + al * AR * 8;                          // this atom-lane's column
  char *adjc = reinterpret_cast<char *>(adj) + al * AR * 8;
  const int n_groups = (a.c1 - a.c0 + A - 1) / A;
  for (int g = blockIdx.x; g < n_groups; g += gridDim.x) {
    const int atom0 = a.c0 + g * A + al * AR;                      // this thread's first atom
    const int n_ok = min(AR, max(0, a.c1 - atom0));                // how many of its atoms exist
    const long long col = atom0 - a.c0;
    __syncthreads();                         // previous group's reads are done (and wsm / psm are filled)
    for (int k = rl; k < a.n_basic; k += R) {
      Vec<AR> m;
#pragma unroll
      for (int r = 0; r < AR; ++r) m.v[r] = r < n_ok ? a.M[tiled_index(a.n_rows, a.mload_k ? a.mload_k[k] : k, col + r)] : 0.0;
      sts<AR>(const_cast<char *>(valc) + (size_t)k * A * 8, m);
    }
    if (a.want_adj)
      for (int k = rl; k < a.n_adj; k += R) {
        Vec<AR> s;
#pragma unroll
        for (int r = 0; r < AR; ++r) s.v[r] = a.adj_init[k];
        sts<AR>(adjc + (size_t)k * A * 8, s);
      }
    if (a.want_adj && a.Sbar) {              // per-atom seeds of a group's cut nodes (after the constant init)
      __syncthreads();
      for (int q = rl; q < a.n_cut; q += R) {
        Vec<AR> s;
#pragma unroll
        for (int r = 0; r < AR; ++r) s.v[r] = r < n_ok ? a.Sbar[tiled_index(a.n_cut_rows, a.cut_row[q], col + r)] : 0.0;
        sts<AR>(adjc + (size_t)a.cut_aslot[q] * A * 8, s);
      }
    }
    __syncthreads();
    Vec<AR> e;
#pragma unroll
    for (int r = 0; r < AR; ++r) e.v[r] = 0.0;
    run_pass<AL, AR, R, false, PS>(fprog, fw, a.nfw, rl, valc, nullptr, const_cast<char *>(valc), a.leaf_seed, e, nullptr,
                                   n_ok, false);
    // ---- energy (stored basis nodes here, elided leaves were added inside the waves) and basis values
    {
      for (int q = rl; q < a.n_eseed; q += R) {
        const Vec<AR> v = lds<AR>(valc + (size_t)a.eseed_slot[q] * A * 8);
        const double sd = a.eseed_val[q];
#pragma unroll
        for (int r = 0; r < AR; ++r) e.v[r] = fma(sd, v.v[r], e.v[r]);
      }
#pragma unroll
      for (int r = 0; r < AR; ++r) esm[(rl * A) + al * AR + r] = e.v[r];
      if (a.B) {        // tiled Bt[b][column]: consecutive threads write consecutive atoms of one b
        const int na = min(A, a.c1 - (a.c0 + g * A));
        for (int i = threadIdx.x; i < na * a.n_basis; i += NT) {
          const int b = i / na, at = i - b * na;
          a.B[tiled_index(a.n_basis, b, g * A + at)] = val[a.basis_slot[b] * A + at];
        }
      }
      __syncthreads();
      if (a.S)                                   // cut values of a group: exported for the top program
        for (int q = rl; q < a.n_cut; q += R) {
          const Vec<AR> v = lds<AR>(valc + (size_t)a.cut_vslot[q] * A * 8);
#pragma unroll
          for (int r = 0; r < AR; ++r)
            if (r < n_ok) a.S[tiled_index(a.n_cut_rows, a.cut_row[q], col + r)] = v.v[r];
        }
      if (rl == 0 && a.write_energy) {           // fixed-order reduction over the R row-lanes
#pragma unroll
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
    double *Gcol = a.G + tiled_index(a.n_rows, 0, col);     // a lane's AR atoms are consecutive columns of one tile
    for (int q = rl; q < a.n_gzero; q += R)
#pragma unroll
      for (int r = 0; r < AR; ++r)
        if (r < n_ok) Gcol[a.gzero_k[q] * kTile + r] = 0.0;
    run_pass<AL, AR, R, true, PS>(bprog, bw, a.nbw, rl, valc, adjc, const_cast<char *>(valc), nullptr, e, Gcol, n_ok, a.g_accum != 0);
    __syncthreads();
    // packed moments that are basis functions themselves (M_{mu,0}): G += xi
    for (int q = rl; q < a.n_gseed; q += R)
#pragma unroll
      for (int r = 0; r < AR; ++r)
        if (r < n_ok) Gcol[a.gseed_k[q] * kTile + r] += a.gseed_val[q];
  }
}

// shared memory: val [n_val][A] + adj [n_adj][A] + energy partials [NT][AR] + wave offsets (<= 1 KB)
// [+ the program when it is staged]
int tree_threads(int AL) { return AL >= 16 ? 512 : (AL == 8 ? 256 : 128); }
int tree_row_lanes(int AL) { return tree_threads(AL) / AL; }
size_t tree_smem_bytes(int n_val, int n_adj, int AL, int AR) {
  return (((size_t)n_val + (size_t)n_adj) * AL * AR * 8 + (size_t)tree_threads(AL) * AR * 8 + 1024 + 15) & ~(size_t)15;
}
constexpr size_t kTreeSmemMax = 225 * 1024;

// Atoms per CTA as (AL, AR): the largest that fits in shared memory, reduced for small systems so
// that the grid still covers the SMs (PAPER.md:35,182 small-system regime).
void tree_pick_shape(int n_val, int n_adj, long long n_atoms, int *AL, int *AR) {
  *AL = 0; *AR = 1;
  static const int shapes[][2] = {{32, 2}, {32, 1}, {16, 1}, {8, 1}, {4, 1}, {2, 1}, {1, 1}};
  for (auto &sh : shapes) {
    if (tree_smem_bytes(n_val, n_adj, sh[0], sh[1]) > kTreeSmemMax) continue;
    const long long A = sh[0] * sh[1];
    if (n_atoms > 0 && A > 4 && (n_atoms + A - 1) / A < 296) continue;   // too few CTAs for 148 SMs
    *AL = sh[0]; *AR = sh[1];
    return;
  }
}

template <int AL, int AR, int NT, bool PS>
static cudaError_t launch_al(const TreeArgs &a0, size_t smem, cudaStream_t st) {
  static bool attr_done = false;
  static int sms = 148;
  if (!attr_done) {
    cudaError_t e = cudaFuncSetAttribute(k_tree<AL, AR, NT, PS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTreeSmemMax);
    if (e != cudaSuccess) return e;
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    attr_done = true;
  }
  const int n = a0.c1 - a0.c0;
  const int groups = (n + AL * AR - 1) / (AL * AR);
  if (groups <= 0) return cudaSuccess;
  int per_sm = 1;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_tree<AL, AR, NT, PS>, NT, smem);
  if (per_sm < 1) per_sm = 1;
  const int grid = groups < sms * per_sm ? groups : sms * per_sm;
  k_tree<AL, AR, NT, PS><<<grid, NT, smem, st>>>(a0);
  count_launch();
  return cudaGetLastError();
}

template <int AL, int AR, int NT>
static cudaError_t launch_ps(TreeArgs a, cudaStream_t st) {
  // stage the program in shared memory when it fits beside the node arrays and the CTA has
  // enough atom groups to amortise the copy
  const size_t base = tree_smem_bytes(a.n_val, a.n_adj, AL, AR);
  const size_t pbytes = ((size_t)a.n_fprog + a.n_bprog) * sizeof(TreeTerm);
  const long long groups = (a.c1 - a.c0 + AL * AR - 1) / (AL * AR);
  if (base + pbytes <= kTreeSmemMax && groups >= 4 * 148) {
    a.prog_smem_off = (int)base;
    return launch_al<AL, AR, NT, true>(a, base + pbytes, st);
  }
  a.prog_smem_off = 0;
  return launch_al<AL, AR, NT, false>(a, base, st);
}

cudaError_t launch_tree(const TreeArgs &a, int AL, int AR, cudaStream_t st) {
  switch (AL * 4 + AR) {
    case 1 * 4 + 1: return launch_ps<1, 1, 128>(a, st);
    case 2 * 4 + 1: return launch_ps<2, 1, 128>(a, st);
    case 4 * 4 + 1: return launch_ps<4, 1, 128>(a, st);
    case 8 * 4 + 1: return launch_ps<8, 1, 256>(a, st);
    case 16 * 4 + 1: return launch_ps<16, 1, 512>(a, st);
    case 32 * 4 + 1: return launch_ps<32, 1, 512>(a, st);
    case 32 * 4 + 2: return launch_ps<32, 2, 512>(a, st);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace mtpb
