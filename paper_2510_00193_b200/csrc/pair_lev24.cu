// K1 / K3 instantiation for the level-24 staircase (NSB=2, NSC=4, block-parallel P=4;
// large systems: the components dealt to 8 warps of a CTA, pair_sliced.cuh).
#include "pair_level.cuh"
namespace mtpb {
PairLevel pair_level_24() { return PairLevelImpl<24, 2, 4, 4, 8>::record(); }
}  // namespace mtpb
