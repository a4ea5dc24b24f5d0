// hr_hop.cu — dispatch of the hopping kernels (H1/H2/H3).
#include "hr_dirac_tiled.cuh"

namespace hr {

// lattices below this many sites fit L2 several times over and are launch-bound: the generic kernel's
// many small CTAs spread better there than one marching CTA per tile
static const double TILED_AUTO_MIN_SITES = 32.0 * 32.0 * 32.0 * 32.0;

int sm_count() {   // of the calling thread's current device (cached per device)
    static std::atomic<int> cache[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { (void)cudaGetLastError(); return 148; }
    int n = cache[dev].load(std::memory_order_relaxed);
    if (n == 0) {
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
            (void)cudaGetLastError();
            n = 148;
        }
        cache[dev].store(n, std::memory_order_relaxed);
    }
    return n;
}

bool tiled_supported(const hr_geom* g) {
    if (g->rep == HR_REP_SU3) return false;     // complex 3 x 3 links: generic kernel only
    TiledPlan pl;
    return tiled_plan(g, 0, 148, pl);     // (whether a tile shape fits does not depend on the SM count)
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

// the launch plan of an operator on this geometry, for tests and diagnostics (hr_kernel_plan)
int kernel_plan(const hr_geom* g, int both, int* info) {
    for (int i = 0; i < 8; ++i) info[i] = 0;
    if (!tiled_chosen(g)) return HR_OK;            // generic kernel: info[0] = 0
    DiracPlan dp;
    if (both == 2 && dirac_plan(g, sm_count(), dp)) {
        const int v[8] = {2, dp.t1, dp.t2, dp.nseg, dp.seglen, dp.nconsumer + 32, (int)dp.smem, dp.nt1 * dp.nt2 * dp.nseg};
        for (int i = 0; i < 8; ++i) info[i] = v[i];
        return HR_OK;
    }
    TiledPlan pl;
    if (!tiled_plan(g, both ? 1 : 0, sm_count(), pl)) return HR_OK;
    size_t smem = pl.smem;      // + the link slots where launch_hop_tiled_l3h uses them (fundamental representation, bare / axpy parity hop)
    const size_t with_links = pl.smem + (size_t)8 * link_chunks(g->prec) * 16 * pl.nconsumer;
    if (HOP_ALINK && !both && g->rep == HR_REP_FUND && with_links <= TILED_SMEM_LIMIT) smem = with_links;
    const int v[8] = {1, pl.t1, pl.t2, pl.nseg, pl.seglen, pl.nconsumer + 32, (int)smem, (both ? 2 : 1) * pl.nt1 * pl.nt2 * pl.nseg};
    for (int i = 0; i < 8; ++i) info[i] = v[i];
    return HR_OK;
}

int run_hop(const hr_geom* g, const HopArgs& a, int epi, cudaStream_t st) {
    const Geo geo = make_geo(g);
    TiledPlan pl;
    // a hop with cut directions (hr_hop_local): tiled open-boundary kernel for the fundamental representation, else generic
    const bool open_ok = a.open_mask == 0 || (g->rep == HR_REP_FUND && !a.both);
    const bool fits = g->kernel != HR_KERNEL_GENERIC && g->rep != HR_REP_SU3 && open_ok && tiled_plan(g, a.both, sm_count(), pl);
    if (g->kernel == HR_KERNEL_TILED && !fits && open_ok) {
        set_error("HR_KERNEL_TILED: lattice %dx%dx%dx%d does not fit the tiled kernel", g->L[0], g->L[1], g->L[2], g->L[3]);
        return HR_EUNSUPPORTED;
    }
    if (fits && tiled_chosen(g)) {
        DiracPlan dp;
        if (a.both && epi == EPI_AXPY && a.phi == a.in && dirac_plan(g, sm_count(), dp)) {   // H3: hr_dirac_tiled.cuh
            if (g->prec == HR_PREC_F64) return launch_dirac_tiled<double>(geo, a, dp, st);
            return launch_dirac_tiled<float>(geo, a, dp, st);
        }
        if (a.open_mask) {
            if (g->prec == HR_PREC_F64) return launch_hop_tiled_open<double>(geo, a, epi, pl, st);
            return launch_hop_tiled_open<float>(geo, a, epi, pl, st);
        }
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
    if (g->rep == HR_REP_SU3) {
        if (g->link_storage == HR_LINKS_COMPRESSED) {     // two rows stored
            if (g->prec == HR_PREC_F64) return launch_hop_generic<double, 3, true, true>(geo, a, epi, st);
            return launch_hop_generic<float, 3, true, true>(geo, a, epi, st);
        }
        if (g->prec == HR_PREC_F64) return launch_hop_generic<double, 3, false, true>(geo, a, epi, st);
        return launch_hop_generic<float, 3, false, true>(geo, a, epi, st);
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
