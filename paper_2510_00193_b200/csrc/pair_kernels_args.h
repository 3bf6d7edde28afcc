// Argument block of the pair kernels K1 / K3 (see pair_kernels.cuh).
#pragma once

namespace mtpb {

// Per-atom arrays of a chunk (M, G, S, dE/dS, B) are tiled: [tile of 128 atoms][row][128].  A thread that owns one
// atom then finds all rows at a fixed 1 KB stride from one base pointer (immediate offsets in the generated K2
// kernels), and 16 or 32 consecutive atoms of one row are still one contiguous segment for K1 / K3.
constexpr int kTile = 128;
#ifdef __CUDACC__
__host__ __device__
#endif
inline unsigned long long tiled_index(int n_rows, int row, long long col) {
  return ((unsigned long long)(col >> 7) * (unsigned long long)n_rows + (unsigned long long)row) * 128ull + (unsigned long long)(col & 127);
}

struct PairArgs {
  const double *pos4;        // [N][4] x, y, z, species (as double)
  const long long *off;      // [N+1]
  const int *idx;            // [nnz] packed neighbour words: j | code << 27 (k_pack_pairs); code 0 = no shift,
                             // else 1 + the index of the image shift in {-1,0,1}^3 order with 0,0,0 moved to the front
  const double *coef;        // [S*S][crow] radial coefficients, block = (z_i*S + z_j), [beta][NMUP]
  const int *kmap;           // [NS][NSLOT] slot -> packed component of the table, or -1
  double *M;                 // K1 out: tiled [tiles][n_rows][128], column = atom - c0 (kTile)
  const double *G;           // K3 in : same layout
  double *d4;                // K3 out (gather mode): [d4_cap][4] records of THIS CHUNK's pairs (index p - off[c0]), or null
  long long d4_cap;          // pairs the chunk's d4 buffer holds; a chunk with more sets flag[1] and drops the excess
  int *flag;                 // device error counters: [0] rejected input pairs, [1] per-pair scratch overflow
  const int *cnt;            // live rows (MTP_OPT_SKIN_LIST): cnt[atom - c0] = entries of the atom's row within R_cut, moved to the
                             // front of the row by k_pack_rows_live; null: the CSR row lengths
  const unsigned short *korig;   // live rows: position in the CSR row of the entry at a compacted position (d4 keeps CSR positions)
  int idx_rel;               // 1: idx holds this chunk's pairs only (index p - off[c0]); 0: the whole list
  long long idx_cap;         // entries idx holds (pairs beyond are treated as absent: their chunk overflowed the scratch)
  double *F;                 // K3 out: [N][3]; atomic mode: every pair is scattered with fp64 atomics; gather mode: F_i += the sum of
                             // the atom's own pairs (the reaction terms come from k_gather_chunk)
  double *wpart;             // K3 out: [gridDim.x][8] virial partials
  int n_rows;                // rows of M / G (n_basic)
  int c0, c1;                // atom range of this chunk
  int n_species, nb, crow;
  int minimg;
  double H[9], Hi[9];        // box rows, inverse (columns of Hi map cartesian -> fractional)
  double r_min, r_cut;
  double inv_width;            // 1 / (R_cut - R_min): the Chebyshev argument by a multiplication, not a division per pair
};

}  // namespace mtpb
