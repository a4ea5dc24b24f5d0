// hr_hop.cu — dispatch of the hopping kernels (H1/H2/H3).
#include "hr_hop_generic.cuh"

namespace hr {

bool tiled_supported(const hr_geom*) { return false; }
bool tiled_chosen(const hr_geom* g) { return g->kernel == HR_KERNEL_TILED && tiled_supported(g); }

int run_hop(const hr_geom* g, const HopArgs& a, int epi, cudaStream_t st) {
    const Geo geo = make_geo(g);
    if (g->kernel == HR_KERNEL_TILED && !tiled_supported(g)) {
        set_error("HR_KERNEL_TILED: lattice %dx%dx%dx%d does not fit the tiled kernel", g->L[0], g->L[1], g->L[2], g->L[3]);
        return HR_EUNSUPPORTED;
    }
    if (g->rep == HR_REP_FUND) {
        if (g->prec == HR_PREC_F64) return launch_hop_generic<double, 2>(geo, a, epi, st);
        return launch_hop_generic<float, 2>(geo, a, epi, st);
    }
    if (epi == EPI_CLOVER_INV || epi == EPI_CLOVER_AXPY) {
        set_error("clover epilogues exist for the fundamental representation only");
        return HR_EUNSUPPORTED;
    }
    if (g->prec == HR_PREC_F64) return launch_hop_generic<double, 3>(geo, a, epi, st);
    return launch_hop_generic<float, 3>(geo, a, epi, st);
}

}  // namespace hr
