// hr_hop_cg.cu — the parity hops that carry a stage of the CG solver in their epilogue (POST_G5_NORM, POST_CG_UPDATE of
// hr_hop_generic.cuh; SURVEY.md §8(f) item 2 "fused dot products and axpys in the hop epilogue").  A translation unit of its own so
// that these instantiations build in parallel with hr_hop.cu.  Tiled kernel for the fundamental representation where hr_hop.cu
// would choose it, the generic kernel for everything else.
#include "hr_hop_tiled.cuh"

namespace hr {

static bool post_tiled(const hr_geom* g, TiledPlan& pl) {
    return g->rep == HR_REP_FUND && tiled_chosen(g) && tiled_plan(g, 0, sm_count(), pl);
}

int hop_post_blocks(const hr_geom* g) {
    TiledPlan pl;
    if (post_tiled(g, pl)) return pl.nt1 * pl.nt2 * pl.nseg;
    return (make_geo(g).Vh + 127) / 128;
}

template <typename T, int EPI>
static int tiled_post(const Geo& geo, const HopArgs& a, int post, const TiledPlan& pl, cudaStream_t st) {
    if (post == POST_G5_NORM) return launch_hop_tiled_epi<T, 2, EPI, false, false, false, POST_G5_NORM>(geo, a, pl, st);
    return launch_hop_tiled_epi<T, 2, EPI, false, false, false, POST_CG_UPDATE>(geo, a, pl, st);
}

int run_hop_post(const hr_geom* g, const HopArgs& a, int epi, int post, cudaStream_t st) {
    if ((epi != EPI_AXPY && epi != EPI_CLOVER_AXPY) || (post != POST_G5_NORM && post != POST_CG_UPDATE) || a.both || a.open_mask) {
        set_error("run_hop_post: epilogue %d / stage %d", epi, post);
        return HR_EINVAL;
    }
    const Geo geo = make_geo(g);
    TiledPlan pl;
    if (post_tiled(g, pl)) {
        if (g->prec == HR_PREC_F64) return epi == EPI_AXPY ? tiled_post<double, EPI_AXPY>(geo, a, post, pl, st) : tiled_post<double, EPI_CLOVER_AXPY>(geo, a, post, pl, st);
        return epi == EPI_AXPY ? tiled_post<float, EPI_AXPY>(geo, a, post, pl, st) : tiled_post<float, EPI_CLOVER_AXPY>(geo, a, post, pl, st);
    }
    const bool f64 = g->prec == HR_PREC_F64;
    if (g->rep == HR_REP_SU3) {
        if (g->link_storage == HR_LINKS_COMPRESSED)
            return f64 ? launch_hop_generic_post<double, 3, true, true>(geo, a, epi, post, st) : launch_hop_generic_post<float, 3, true, true>(geo, a, epi, post, st);
        return f64 ? launch_hop_generic_post<double, 3, false, true>(geo, a, epi, post, st) : launch_hop_generic_post<float, 3, false, true>(geo, a, epi, post, st);
    }
    if (g->rep == HR_REP_FUND) return f64 ? launch_hop_generic_post<double, 2, false, false>(geo, a, epi, post, st) : launch_hop_generic_post<float, 2, false, false>(geo, a, epi, post, st);
    if (g->link_storage == HR_LINKS_ONTHEFLY)
        return f64 ? launch_hop_generic_post<double, 3, true, false>(geo, a, epi, post, st) : launch_hop_generic_post<float, 3, true, false>(geo, a, epi, post, st);
    return f64 ? launch_hop_generic_post<double, 3, false, false>(geo, a, epi, post, st) : launch_hop_generic_post<float, 3, false, false>(geo, a, epi, post, st);
}

}  // namespace hr
