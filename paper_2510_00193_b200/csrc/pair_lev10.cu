// K1 / K3 instantiation for the level-10 staircase (NSB=1, NSC=1, block-parallel P=8;
// large systems: the components dealt to 4 warps of a CTA, pair_sliced.cuh).
#include "pair_level.cuh"
namespace mtpb {
PairLevel pair_level_10() { return PairLevelImpl<10, 1, 1, 8, 4>::record(); }
}  // namespace mtpb
