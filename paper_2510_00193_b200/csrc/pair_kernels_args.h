// Argument block of the pair kernels K1 / K3 (see pair_kernels.cuh).
#pragma once

namespace mtpb {

struct PairArgs {
  const double *pos4;        // [N][4] x, y, z, species (as double)
  const long long *off;      // [N+1]
  const int *idx;            // [nnz] packed neighbour words: j | code << 27 (k_pack_pairs); code 0 = no shift,
                             // else 1 + the index of the image shift in {-1,0,1}^3 order with 0,0,0 moved to the front
  const double *coef;        // [S*S][crow] radial coefficients, block = (z_i*S + z_j), [beta][NMUP]
  const int *kmap;           // [NS][NSLOT] slot -> packed component of the table, or -1
  double *M;                 // K1 out: [n_basic][ldm], column = atom - c0
  const double *G;           // K3 in : [n_basic][ldm]
  double *d4;                // K3 out (gather mode): [nnz][4], or null
  double *F;                 // K3 out (atomic mode): [N][3], or null
  double *wpart;             // K3 out: [gridDim.x][8] virial partials
  long long ldm;
  int c0, c1;                // atom range of this chunk
  int n_species, nb, crow;
  int minimg;
  double H[9], Hi[9];        // box rows, inverse (columns of Hi map cartesian -> fractional)
  double r_min, r_cut;
};

}  // namespace mtpb
