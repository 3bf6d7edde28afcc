// K1 / K3 instantiation for the level-20 staircase (NSB=2, NSC=2, block-parallel P=8).
#include "pair_level.cuh"
namespace mtpb {
PairLevel pair_level_20() { return PairLevelImpl<20, 2, 2, 8>::record(); }
}  // namespace mtpb
