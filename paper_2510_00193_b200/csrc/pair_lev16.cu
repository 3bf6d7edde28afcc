// K1 / K3 instantiation for the level-16 staircase (NSB=1, NSC=2, block-parallel P=8;
// large systems: the components dealt to 4 warps of a CTA, pair_sliced.cuh).
#include "pair_level.cuh"
namespace mtpb {
PairLevel pair_level_16() { return PairLevelImpl<16, 1, 2, 8, 4>::record(); }
}  // namespace mtpb
