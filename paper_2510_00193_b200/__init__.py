"""B200-native Moment Tensor Potential hot path (arxiv 2510.00193): CUDA kernels behind the
C ABI of include/mtp_b200.h plus this thin ctypes binding.  No CPU fallback."""
from .binding import (Table, Potential, MtpError, launch_count, peak_dfma, neighbors_build, neighbors_build_static, dump_selected, NB_STATIC_MAX_ATOMS, LIB_PATH, EXPORTS,
                      OK, EINVAL, ESIZE, EBOX, ECUDA, EUNSUP, ENOMEM,
                      OPT_CHUNK_ATOMS, OPT_FORCE_MODE, OPT_VARIANT, OPT_PROFILE, OPT_TREE_CODEGEN, INFO_TREE_KERNELS,
                      INFO_TREE_PROGRAMS, INFO_INPUT_ERRORS, INFO_SCRATCH_OVERFLOW, OPT_CHUNK_PAIRS, OPT_SKIN_LIST,
                      FORCE_GATHER, FORCE_ATOMIC, FORCE_AUTO,
                      VARIANT_AUTO, VARIANT_THREAD, VARIANT_BLOCK)
