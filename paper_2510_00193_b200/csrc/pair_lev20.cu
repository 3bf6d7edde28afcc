// K1 / K3 instantiation for the level-20 staircase (NSB=2, NSC=2, block-parallel P=8;
// large systems: the components dealt to 8 warps of a CTA, pair_sliced.cuh).
#include "pair_level.cuh"
namespace mtpb {
PairLevel pair_level_20() { return PairLevelImpl<20, 2, 2, 8, 8>::record(); }
}  // namespace mtpb
