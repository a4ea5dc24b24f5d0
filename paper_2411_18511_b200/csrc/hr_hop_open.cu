// hr_hop_open.cu — the tiled hop with open boundaries (OPEN = true instantiations of hop_tiled_kernel): the interior kernel of
// hr_hop_local for the fundamental representation.  A translation unit of its own so that it builds in parallel.
#include "hr_hop_tiled.cuh"

namespace hr {

template <typename T>
int launch_hop_tiled_open(const Geo& g, const HopArgs& a, int epi, const TiledPlan& pl, cudaStream_t st) {
    switch (epi) {
        case EPI_NONE: return launch_hop_tiled_epi<T, 2, EPI_NONE, false, false, true>(g, a, pl, st);
        case EPI_AXPY: return launch_hop_tiled_epi<T, 2, EPI_AXPY, false, false, true>(g, a, pl, st);
        case EPI_CLOVER_INV: return launch_hop_tiled_epi<T, 2, EPI_CLOVER_INV, false, false, true>(g, a, pl, st);
        case EPI_CLOVER_AXPY: return launch_hop_tiled_epi<T, 2, EPI_CLOVER_AXPY, false, false, true>(g, a, pl, st);
        default: set_error("unknown epilogue %d", epi); return HR_EINVAL;
    }
}
template int launch_hop_tiled_open<double>(const Geo&, const HopArgs&, int, const TiledPlan&, cudaStream_t);
template int launch_hop_tiled_open<float>(const Geo&, const HopArgs&, int, const TiledPlan&, cudaStream_t);

}  // namespace hr
