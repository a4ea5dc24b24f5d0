// hr_hop.cu — dispatch of the hopping kernels (H1/H2/H3).
#include "hr_hop_tiled.cuh"

namespace hr {

// lattices below this many sites fit L2 several times over and are launch-bound: the generic kernel's
// many small CTAs spread better there than one marching CTA per tile
static const double TILED_AUTO_MIN_SITES = 32.0 * 32.0 * 32.0 * 32.0;

static int sm_count() {   // of the calling thread's current device (cached per device)
    static int cache[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { (void)cudaGetLastError(); return 148; }
    if (cache[dev] == 0) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
            (void)cudaGetLastError();
            n = 148;
        }
        cache[dev] = n;
    }
    return cache[dev];
}

bool tiled_supported(const hr_geom* g) {
    TiledPlan pl;
    return tiled_plan(g, 0, 148, pl);
}

bool tiled_chosen(const hr_geom* g) {
    if (g->kernel == HR_KERNEL_GENERIC || !tiled_supported(g)) return false;
    if (g->kernel == HR_KERNEL_TILED) return true;
    // adjoint rows are 1.5x longer: the 2x4 tile then takes > 200 KiB of shared memory, which starves the L1 the link
    // loads go through; measured slower than the generic kernel at every size (L = 16..40), so AUTO keeps generic
    if (g->rep == HR_REP_ADJ) return false;
    const double v = (double)g->L[0] * g->L[1] * g->L[2] * g->L[3];
    return v >= TILED_AUTO_MIN_SITES;
}

int run_hop(const hr_geom* g, const HopArgs& a, int epi, cudaStream_t st) {
    const Geo geo = make_geo(g);
    if (g->kernel == HR_KERNEL_TILED && !tiled_supported(g)) {
        set_error("HR_KERNEL_TILED: lattice %dx%dx%dx%d does not fit the tiled kernel", g->L[0], g->L[1], g->L[2], g->L[3]);
        return HR_EUNSUPPORTED;
    }
    if (tiled_chosen(g)) {
        TiledPlan pl;
        tiled_plan(g, a.both, sm_count(), pl, a.both && epi == EPI_AXPY && a.phi == a.in);
        if (g->rep == HR_REP_FUND) {
            if (g->prec == HR_PREC_F64) return launch_hop_tiled<double, 2>(geo, a, epi, pl, st);
            return launch_hop_tiled<float, 2>(geo, a, epi, pl, st);
        }
        if (g->link_storage == HR_LINKS_ONTHEFLY) {
            if (g->prec == HR_PREC_F64) return launch_hop_tiled<double, 3, true>(geo, a, epi, pl, st);
            return launch_hop_tiled<float, 3, true>(geo, a, epi, pl, st);
        }
        if (g->prec == HR_PREC_F64) return launch_hop_tiled<double, 3>(geo, a, epi, pl, st);
        return launch_hop_tiled<float, 3>(geo, a, epi, pl, st);
    }
    if (g->rep == HR_REP_FUND) {
        if (g->prec == HR_PREC_F64) return launch_hop_generic<double, 2>(geo, a, epi, st);
        return launch_hop_generic<float, 2>(geo, a, epi, st);
    }
    if (g->link_storage == HR_LINKS_ONTHEFLY) {
        if (g->prec == HR_PREC_F64) return launch_hop_generic<double, 3, true>(geo, a, epi, st);
        return launch_hop_generic<float, 3, true>(geo, a, epi, st);
    }
    if (g->prec == HR_PREC_F64) return launch_hop_generic<double, 3>(geo, a, epi, st);
    return launch_hop_generic<float, 3>(geo, a, epi, st);
}

}  // namespace hr
