// K1 / K3 instantiation for the level-10 staircase (NSB=1, NSC=1, block-parallel P=8).
#include "pair_level.cuh"
namespace mtpb {
PairLevel pair_level_10() { return PairLevelImpl<10, 1, 1, 8>::record(); }
}  // namespace mtpb
