// K1 / K3 instantiation for the level-16 staircase (NSB=1, NSC=2, block-parallel P=8).
#include "pair_level.cuh"
namespace mtpb {
PairLevel pair_level_16() { return PairLevelImpl<16, 1, 2, 8>::record(); }
}  // namespace mtpb
