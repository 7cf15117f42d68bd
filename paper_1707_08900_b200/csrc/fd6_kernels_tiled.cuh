// fd6_kernels_tiled.cuh — FD_VARIANT_TILED: TMA-staged xy tiles in shared memory with a register sliding
// window along z.  Placeholder until the tiled kernels land: reports "unsupported" so
// FD_VARIANT_AUTO resolves to the direct kernels.
#pragma once
#include "fd6_common.cuh"

namespace fd6 {

struct TiledState {
    bool ready = false;
};

inline bool tiled_supported(const Geom&, int /*dtype*/) { return false; }
inline const char* tiled_error() { return "tiled variant not built"; }
inline int tiled_prepare(TiledState&, const Geom&, int, void*, void*, void*) { return 4 /*FD_EUNSUPPORTED*/; }
inline void tiled_release(TiledState&) {}

template <class T, class Scope, class Halo>
int tiled_substep(TiledState&, int, int, const T*, T*, T*, T*, const Geom&, const Coef<T>&, const Sub<T>&, cudaStream_t,
                  Scope, Halo) {
    return 4;
}

}  // namespace fd6
