// fd6_tiled_inst.cu — one translation unit of tiled-kernel instantiations: value type FD6_INST_T (float, double, V2),
// FD6_INST_FORCE (false, true) and tile shape FD6_INST_SHAPE (0 wide, 1 tall), given on the command line by build.py,
// which compiles the ten units in parallel.
#include "fd6_kernels_tiled.cuh"

#if !defined(FD6_INST_T) || !defined(FD6_INST_FORCE) || !defined(FD6_INST_SHAPE)
#error "build.py defines FD6_INST_T, FD6_INST_FORCE and FD6_INST_SHAPE"
#endif

namespace fd6 {
template struct TiledTU<FD6_INST_T, FD6_INST_FORCE, FD6_INST_SHAPE>;
}
