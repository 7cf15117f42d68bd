// fd6_tiled_inst.cu — one translation unit of tiled-kernel instantiations: value type FD6_INST_T (float, double, V2)
// and FD6_INST_FORCE (false, true), given on the command line by build.py, which compiles the six units in parallel.
#include "fd6_kernels_tiled.cuh"

#if !defined(FD6_INST_T) || !defined(FD6_INST_FORCE)
#error "build.py defines FD6_INST_T and FD6_INST_FORCE"
#endif

namespace fd6 {
template struct TiledTU<FD6_INST_T, FD6_INST_FORCE>;
}
