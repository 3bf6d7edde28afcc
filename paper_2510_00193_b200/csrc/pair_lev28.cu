// K1 / K3 instantiation for the level-28 staircase (NSB=4, NSC=4, block-parallel P=2).
#include "pair_level.cuh"
namespace mtpb {
PairLevel pair_level_28() { return PairLevelImpl<28, 4, 4, 2>::record(); }
}  // namespace mtpb
