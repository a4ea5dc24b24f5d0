// hr_api.cu — the extern "C" entry points of libhr_dslash (include/hr_dslash.h): argument checks,
// size queries, the work model M1, composition of the operators from the kernels, host-buffer path.
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstring>

#include "hr_hop_generic.cuh"

namespace hr {

// hr_fields.cu
int permute_chunks(bool pack, const Geo& g, int NI, int NCH, int SRC, const void* src, void* dst, cudaStream_t st);
int rebuild_second_row(const Geo& g, int prec, void* canon, cudaStream_t st);
int permute_adj(bool pack, const Geo& g, int prec, const void* src, void* dst, cudaStream_t st, bool complex_entries = false, bool two_rows = false);
int run_represent(const Geo& g, int prec, const void* ufund, void* uadj, cudaStream_t st);
int run_represent_antisym_su3(const Geo& g, int prec, bool tworows, const void* ufund, void* urep, cudaStream_t st);
int run_clover_build(const Geo& g, int prec, double diag, double csw, int expo, const void* ufund, void* fwd, void* inv, cudaStream_t st);
int run_clover_build_adj(const Geo& g, int prec, double diag, double csw, int expo, const void* ufund, void* fwd, void* inv, cudaStream_t st);
int run_clover_build_c3(const Geo& g, int prec, bool two_rows, double diag, double csw, int expo, const void* gauge, void* fwd, void* inv, cudaStream_t st);
int run_clover_apply(const Geo& g, int rep, int prec, int parity, const void* blocks, const void* in, void* out, cudaStream_t st);
int run_count_nonfinite(int prec, const void* x, size_t bytes, unsigned long long* count_dev, cudaStream_t st);

// hr_halo.cu
int run_halo_pack(const hr_geom* hg, const int* split, int par, const void* gauge, const void* in_half, void* const* face_out, cudaStream_t st);
int run_halo_boundary(const hr_geom* hg, const int* split, const HopArgs& a, int epi, const void* const* face_in, cudaStream_t st);
size_t halo_face_bytes(const hr_geom* hg, int mu);

// hr_solver.cu
size_t cg_workspace_bytes(const hr_geom* g);
int run_cg(const hr_geom* g, double m0, const void* u, const void* cf, const void* ci, const void* b, void* x, void* workspace, double tol,
           int max_iter, int check_every, int* iters_out, double* relres_out, cudaStream_t st);
size_t cg_mixed_workspace_bytes(const hr_geom* g);
int run_cg_mixed(const hr_geom* g, double m0, const void* u64, const void* u32, const void* cf64, const void* ci64, const void* cf32, const void* ci32,
                 const void* b, void* x, void* workspace, double tol, double inner_tol,
                 int max_outer, int max_inner, int check_every, int* outer_out, int* inner_out, double* relres_out, cudaStream_t st);

static thread_local char g_err[512] = "";
static std::atomic<unsigned long long> g_launches{0};

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}
void count_launch(int n) { g_launches.fetch_add((unsigned long long)n, std::memory_order_relaxed); }
int check_launch(const char* what) {
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        set_error("%s: %s", what, cudaGetErrorString(e));
        return HR_ECUDA;
    }
    return HR_OK;
}

static int check_geom(const hr_geom* g) {
    if (!geom_ok(g)) {
        set_error("invalid hr_geom (extents must be even and >= 2, volume < 2e9, enums in range)");
        return HR_EINVAL;
    }
    return HR_OK;
}
static int check_ptr(const void* p, const char* name) {
    if (!p) {
        set_error("%s is NULL", name);
        return HR_EINVAL;
    }
    if (reinterpret_cast<uintptr_t>(p) & 15) {
        set_error("%s is not 16-byte aligned", name);
        return HR_EALIGN;
    }
    return HR_OK;
}
static int check_no_su3(const hr_geom* g, const char* what) {
    if (g->rep == HR_REP_SU3) { set_error("%s: not available for HR_REP_SU3", what); return HR_EUNSUPPORTED; }
    return HR_OK;
}
static int check_links(const hr_geom* g) {
    if (g->rep == HR_REP_FUND && g->link_storage != HR_LINKS_COMPRESSED) {
        set_error("HR_LINKS_FULL is a byte-model option only; kernels read HR_LINKS_COMPRESSED fundamental links");
        return HR_EUNSUPPORTED;
    }
    return HR_OK;
}
static bool overlap(const void* a, size_t na, const void* b, size_t nb) {
    const char* x = (const char*)a;
    const char* y = (const char*)b;
    return x < y + nb && y < x + na;
}
#define HR_TRY(expr)                 \
    do {                             \
        int rc_ = (expr);            \
        if (rc_ != HR_OK) return rc_; \
    } while (0)

static size_t half_spinor_bytes(const hr_geom* g) {
    const Geo geo = make_geo(g);
    return (size_t)geo.Vh * spinor_chunks(g->rep, g->prec) * 16;
}

}  // namespace hr

using namespace hr;

extern "C" {

size_t hr_spinor_bytes(const hr_geom* g, int parity) {
    if (!geom_ok(g) || parity < HR_EVEN || parity > HR_BOTH) return 0;
    return half_spinor_bytes(g) * (parity == HR_BOTH ? 2 : 1);
}

size_t hr_gauge_bytes(const hr_geom* g, int rep) {
    if (!geom_ok(g) || (rep != HR_REP_FUND && rep != HR_REP_ADJ && rep != HR_REP_SU3)) return 0;
    const Geo geo = make_geo(g);
    const size_t links = 8 * (size_t)geo.Vh;
    if (rep == HR_REP_FUND) return links * link_chunks(g->prec) * 16;
    return links * (rep == HR_REP_SU3 ? (g->link_storage == HR_LINKS_COMPRESSED ? 12 : 18) : 9) * real_bytes(g->prec);
}

size_t hr_clover_bytes(const hr_geom* g) {
    if (!geom_ok(g)) return 0;
    const Geo geo = make_geo(g);
    return 2 * (size_t)geo.Vh * clover_chunks(g->prec, g->rep) * 16;
}

size_t hr_canonical_spinor_bytes(const hr_geom* g) {
    if (!geom_ok(g)) return 0;
    const Geo geo = make_geo(g);
    return 2 * (size_t)geo.Vh * 8 * ncolour(g->rep) * real_bytes(g->prec);
}

size_t hr_canonical_gauge_bytes(const hr_geom* g, int rep) {
    if (!geom_ok(g) || (rep != HR_REP_FUND && rep != HR_REP_ADJ && rep != HR_REP_SU3)) return 0;
    const Geo geo = make_geo(g);
    return 8 * (size_t)geo.Vh * (rep == HR_REP_FUND ? 8 : rep == HR_REP_SU3 ? 18 : 9) * real_bytes(g->prec);
}

size_t hr_canonical_clover_bytes(const hr_geom* g) {
    if (!geom_ok(g)) return 0;
    const Geo geo = make_geo(g);
    const size_t d = 2 * (size_t)ncolour(g->rep);
    return 2 * (size_t)geo.Vh * 2 * d * d * real_bytes(g->prec);
}

// ---------------------------------------------------------------- pack / unpack
int hr_pack_spinor(const hr_geom* g, const void* canon, void* dev, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_ptr(canon, "canon")); HR_TRY(check_ptr(dev, "dev"));
    const int nch = spinor_chunks(g->rep, g->prec);
    return permute_chunks(true, make_geo(g), 1, nch, nch, canon, dev, (cudaStream_t)stream);
}
int hr_unpack_spinor(const hr_geom* g, const void* dev, void* canon, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_ptr(canon, "canon")); HR_TRY(check_ptr(dev, "dev"));
    const int nch = spinor_chunks(g->rep, g->prec);
    return permute_chunks(false, make_geo(g), 1, nch, nch, dev, canon, (cudaStream_t)stream);
}
int hr_pack_gauge(const hr_geom* g, int rep, const void* canon, void* dev, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_ptr(canon, "canon")); HR_TRY(check_ptr(dev, "dev"));
    if (rep == HR_REP_FUND) {
        if (g->link_storage == HR_LINKS_FULL) { set_error("only HR_LINKS_COMPRESSED fundamental links are stored"); return HR_EUNSUPPORTED; }
        const int lch = link_chunks(g->prec);
        return permute_chunks(true, make_geo(g), 4, lch, 2 * lch, canon, dev, (cudaStream_t)stream);
    }
    if (rep == HR_REP_ADJ) return permute_adj(true, make_geo(g), g->prec, canon, dev, (cudaStream_t)stream);
    if (rep == HR_REP_SU3) return permute_adj(true, make_geo(g), g->prec, canon, dev, (cudaStream_t)stream, true, g->link_storage == HR_LINKS_COMPRESSED);
    set_error("unknown representation %d", rep);
    return HR_EINVAL;
}
int hr_unpack_gauge(const hr_geom* g, int rep, const void* dev, void* canon, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_ptr(canon, "canon")); HR_TRY(check_ptr(dev, "dev"));
    if (rep == HR_REP_FUND) {
        if (g->link_storage == HR_LINKS_FULL) { set_error("only HR_LINKS_COMPRESSED fundamental links are stored"); return HR_EUNSUPPORTED; }
        const int lch = link_chunks(g->prec);
        const Geo geo = make_geo(g);
        HR_TRY(permute_chunks(false, geo, 4, lch, 2 * lch, dev, canon, (cudaStream_t)stream));
        return rebuild_second_row(geo, g->prec, canon, (cudaStream_t)stream);
    }
    if (rep == HR_REP_ADJ) return permute_adj(false, make_geo(g), g->prec, dev, canon, (cudaStream_t)stream);
    if (rep == HR_REP_SU3) return permute_adj(false, make_geo(g), g->prec, dev, canon, (cudaStream_t)stream, true, g->link_storage == HR_LINKS_COMPRESSED);
    set_error("unknown representation %d", rep);
    return HR_EINVAL;
}
int hr_pack_clover(const hr_geom* g, const void* canon, void* dev, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_ptr(canon, "canon")); HR_TRY(check_ptr(dev, "dev"));
    const int cch = clover_chunks(g->prec, g->rep);
    return permute_chunks(true, make_geo(g), 1, cch, cch, canon, dev, (cudaStream_t)stream);
}
int hr_unpack_clover(const hr_geom* g, const void* dev, void* canon, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_ptr(canon, "canon")); HR_TRY(check_ptr(dev, "dev"));
    const int cch = clover_chunks(g->prec, g->rep);
    return permute_chunks(false, make_geo(g), 1, cch, cch, dev, canon, (cudaStream_t)stream);
}

// ---------------------------------------------------------------- R1
int hr_represent_gauge(const hr_geom* g, const void* u_fund, void* u_adj, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_no_su3(g, "hr_represent_gauge")); HR_TRY(check_ptr(u_fund, "u_fund")); HR_TRY(check_ptr(u_adj, "u_adj"));
    if (g->link_storage == HR_LINKS_FULL) { set_error("only HR_LINKS_COMPRESSED fundamental links are stored"); return HR_EUNSUPPORTED; }
    return run_represent(make_geo(g), g->prec, u_fund, u_adj, (cudaStream_t)stream);
}

int hr_represent_gauge_antisym(const hr_geom* g, const void* u_fund, void* u_rep, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_ptr(u_fund, "u_fund")); HR_TRY(check_ptr(u_rep, "u_rep"));
    if (g->rep != HR_REP_SU3) { set_error("hr_represent_gauge_antisym: complex 3 x 3 links only (g->rep must be HR_REP_SU3)"); return HR_EUNSUPPORTED; }
    if (overlap(u_fund, hr_gauge_bytes(g, HR_REP_SU3), u_rep, hr_gauge_bytes(g, HR_REP_SU3))) { set_error("hr_represent_gauge_antisym: u_rep aliases u_fund"); return HR_EINVAL; }
    return run_represent_antisym_su3(make_geo(g), g->prec, g->link_storage == HR_LINKS_COMPRESSED, u_fund, u_rep, (cudaStream_t)stream);
}

// ---------------------------------------------------------------- H3
int hr_dirac_apply(const hr_geom* g, double m0, const void* u, const void* psi, void* out, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_links(g));
    HR_TRY(check_ptr(u, "u")); HR_TRY(check_ptr(psi, "psi")); HR_TRY(check_ptr(out, "out"));
    const size_t full = 2 * half_spinor_bytes(g);
    if (overlap(psi, full, out, full)) { set_error("hr_dirac_apply: out aliases psi (gather operation)"); return HR_EINVAL; }
    HopArgs a;
    a.gauge = u; a.in = psi; a.out = out; a.phi = psi; a.clover = nullptr;
    a.a = 4.0 + m0; a.c = -0.5; a.parity = 0; a.both = 1;
    return run_hop(g, a, EPI_AXPY, (cudaStream_t)stream);
}

int hr_dirac_clover_apply(const hr_geom* g, const void* u, const void* clover_fwd, const void* psi, void* out, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_links(g));
    HR_TRY(check_ptr(u, "u")); HR_TRY(check_ptr(clover_fwd, "clover_fwd")); HR_TRY(check_ptr(psi, "psi")); HR_TRY(check_ptr(out, "out"));
    const size_t full = 2 * half_spinor_bytes(g);
    if (overlap(psi, full, out, full)) { set_error("hr_dirac_clover_apply: out aliases psi (gather operation)"); return HR_EINVAL; }
    HopArgs a;
    a.gauge = u; a.in = psi; a.out = out; a.phi = psi; a.clover = clover_fwd;
    a.a = 1.0; a.c = -0.5; a.parity = 0; a.both = 1;
    return run_hop(g, a, EPI_CLOVER_AXPY, (cudaStream_t)stream);
}

// ---------------------------------------------------------------- H1 / E1 / E2
int hr_dirac_eo_apply(const hr_geom* g, int op, double m0, const void* u, const void* clover_fwd,
                      const void* clover_inv, const void* in, void* out, void* tmp, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_links(g));
    HR_TRY(check_ptr(u, "u")); HR_TRY(check_ptr(in, "in")); HR_TRY(check_ptr(out, "out"));
    const size_t half = half_spinor_bytes(g);
    if (overlap(in, half, out, half)) { set_error("hr_dirac_eo_apply: out aliases in (gather operation)"); return HR_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    HopArgs a;
    a.gauge = u; a.phi = nullptr; a.clover = nullptr; a.a = 0.0; a.c = 1.0; a.both = 0;
    if (op == HR_EO_HOP_OE || op == HR_EO_HOP_EO) {
        a.in = in; a.out = out; a.parity = (op == HR_EO_HOP_OE) ? HR_ODD : HR_EVEN;
        return run_hop(g, a, EPI_NONE, st);
    }
    if (op != HR_EO_DHAT) { set_error("hr_dirac_eo_apply: unknown op %d", op); return HR_EINVAL; }
    HR_TRY(check_ptr(tmp, "tmp"));
    if (overlap(tmp, half, in, half) || overlap(tmp, half, out, half)) { set_error("hr_dirac_eo_apply: tmp aliases in or out"); return HR_EINVAL; }
    const bool clover = clover_fwd || clover_inv;
    if (clover) {
        if (!clover_fwd || !clover_inv) { set_error("hr_dirac_eo_apply: clover_fwd and clover_inv must both be given"); return HR_EINVAL; }
        HR_TRY(check_ptr(clover_fwd, "clover_fwd")); HR_TRY(check_ptr(clover_inv, "clover_inv"));
            // E2: tmp_o = A_oo^-1 H_oe in_e ;  out_e = A_ee in_e - 1/4 H_eo tmp_o
        a.in = in; a.out = tmp; a.parity = HR_ODD; a.clover = clover_inv;
        HR_TRY(run_hop(g, a, EPI_CLOVER_INV, st));
        a.in = tmp; a.out = out; a.parity = HR_EVEN; a.clover = clover_fwd; a.phi = in; a.c = -0.25;
        return run_hop(g, a, EPI_CLOVER_AXPY, st);
    }
    // E1: tmp_o = H_oe in_e ;  out_e = (4+m0) in_e - H_eo tmp_o / (4 (4+m0))
    const double d = 4.0 + m0;
    if (d == 0.0) { set_error("hr_dirac_eo_apply: 4+m0 = 0, D_oo is singular"); return HR_EINVAL; }
    a.in = in; a.out = tmp; a.parity = HR_ODD;
    HR_TRY(run_hop(g, a, EPI_NONE, st));
    a.in = tmp; a.out = out; a.parity = HR_EVEN; a.phi = in; a.a = d; a.c = -1.0 / (4.0 * d);
    return run_hop(g, a, EPI_AXPY, st);
}

// ---------------------------------------------------------------- sharded hop
size_t hr_halo_face_bytes(const hr_geom* g, int mu) {
    if (!geom_ok(g) || mu < 0 || mu > 3) return 0;
    return halo_face_bytes(g, mu);
}

static int check_decomp(const hr_decomp* d) {
    if (!d) { set_error("hr_decomp is NULL"); return HR_EINVAL; }
    return HR_OK;
}

int hr_halo_pack(const hr_geom* g, const hr_decomp* d, int in_parity, const void* u, const void* in_half, void* const* face_out, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_links(g)); HR_TRY(check_decomp(d));
    if (in_parity != HR_EVEN && in_parity != HR_ODD) { set_error("hr_halo_pack: in_parity %d", in_parity); return HR_EINVAL; }
    HR_TRY(check_ptr(u, "u")); HR_TRY(check_ptr(in_half, "in_half"));
    if (!face_out) { set_error("hr_halo_pack: face_out is NULL"); return HR_EINVAL; }
    for (int mu = 0; mu < 4; ++mu)
        if (d->split[mu]) { HR_TRY(check_ptr(face_out[2 * mu], "face_out (down)")); HR_TRY(check_ptr(face_out[2 * mu + 1], "face_out (up)")); }
    return run_halo_pack(g, d->split, in_parity, u, in_half, face_out, (cudaStream_t)stream);
}

// phases: 1 = interior kernel, 2 = boundary kernels, 3 = both
static int hop_local_phases(int phases, const hr_geom* g, const hr_decomp* d, int out_parity, int epi, double a, double c, const void* u,
                            const void* clover, const void* in_half, const void* phi_half, void* out_half, const void* const* face_in, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_links(g)); HR_TRY(check_decomp(d));
    if (out_parity != HR_EVEN && out_parity != HR_ODD) { set_error("hr_hop_local: out_parity %d", out_parity); return HR_EINVAL; }
    if (epi < HR_EPI_NONE || epi > HR_EPI_CLOVER_AXPY) { set_error("hr_hop_local: unknown epilogue %d", epi); return HR_EINVAL; }
    HR_TRY(check_ptr(u, "u")); HR_TRY(check_ptr(out_half, "out_half"));
    if (phases & 1) HR_TRY(check_ptr(in_half, "in_half"));
    if ((phases & 1) && (epi == HR_EPI_AXPY || epi == HR_EPI_CLOVER_AXPY)) HR_TRY(check_ptr(phi_half, "phi_half"));
    if (epi == HR_EPI_CLOVER_INV || epi == HR_EPI_CLOVER_AXPY) HR_TRY(check_ptr(clover, "clover"));
    const size_t half = half_spinor_bytes(g);
    if ((phases & 1) && overlap(in_half, half, out_half, half)) { set_error("hr_hop_local: out aliases in (gather operation)"); return HR_EINVAL; }
    int mask = 0;
    for (int mu = 0; mu < 4; ++mu)
        if (d->split[mu]) {
            if (phases & 2) {
                if (!face_in) { set_error("hr_hop_local: face_in is NULL"); return HR_EINVAL; }
                HR_TRY(check_ptr(face_in[2 * mu], "face_in (down face of the +mu neighbour)"));
                HR_TRY(check_ptr(face_in[2 * mu + 1], "face_in (up face of the -mu neighbour)"));
            }
            mask |= 1 << mu;
        }
    HopArgs h;
    h.gauge = u; h.in = in_half; h.out = out_half; h.phi = phi_half; h.clover = clover;
    h.a = a; h.c = epi == HR_EPI_NONE ? 1.0 : c; h.parity = out_parity; h.both = 0; h.open_mask = mask;
    if (phases & 1) HR_TRY(run_hop(g, h, epi, (cudaStream_t)stream));
    if ((phases & 2) && mask) HR_TRY(run_halo_boundary(g, d->split, h, epi, face_in, (cudaStream_t)stream));
    return HR_OK;
}

int hr_hop_local(const hr_geom* g, const hr_decomp* d, int out_parity, int epi, double a, double c, const void* u, const void* clover,
                 const void* in_half, const void* phi_half, void* out_half, const void* const* face_in, void* stream) {
    return hop_local_phases(3, g, d, out_parity, epi, a, c, u, clover, in_half, phi_half, out_half, face_in, stream);
}

int hr_hop_local_interior(const hr_geom* g, const hr_decomp* d, int out_parity, int epi, double a, double c, const void* u, const void* clover,
                          const void* in_half, const void* phi_half, void* out_half, void* stream) {
    return hop_local_phases(1, g, d, out_parity, epi, a, c, u, clover, in_half, phi_half, out_half, nullptr, stream);
}

int hr_hop_local_boundary(const hr_geom* g, const hr_decomp* d, int out_parity, int epi, double c, const void* u, const void* clover,
                          void* out_half, const void* const* face_in, void* stream) {
    return hop_local_phases(2, g, d, out_parity, epi, 0.0, c, u, clover, nullptr, nullptr, out_half, face_in, stream);
}

// ---------------------------------------------------------------- C1 / C2 / C3
static int clover_build_any(const hr_geom* g, double m0, double csw, int expo, const void* u_fund, void* clover_fwd, void* clover_inv, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_ptr(u_fund, "u_fund"));
    if (g->rep != HR_REP_SU3 && g->link_storage == HR_LINKS_FULL) { set_error("only HR_LINKS_COMPRESSED fundamental links are stored"); return HR_EUNSUPPORTED; }
    if (!clover_fwd && !clover_inv) { set_error("hr_clover_build: nothing to build"); return HR_EINVAL; }
    if (4.0 + m0 == 0.0) { set_error("hr_clover_build: 4+m0 = 0"); return HR_EINVAL; }
    if (clover_fwd) HR_TRY(check_ptr(clover_fwd, "clover_fwd"));
    if (clover_inv) HR_TRY(check_ptr(clover_inv, "clover_inv"));
    if (g->rep == HR_REP_SU3)     // u_fund is then the SU(3) gauge field itself (all three rows, or two with HR_LINKS_COMPRESSED)
        return run_clover_build_c3(make_geo(g), g->prec, g->link_storage == HR_LINKS_COMPRESSED, 4.0 + m0, csw, expo, u_fund, clover_fwd, clover_inv, (cudaStream_t)stream);
    if (g->rep == HR_REP_ADJ) return run_clover_build_adj(make_geo(g), g->prec, 4.0 + m0, csw, expo, u_fund, clover_fwd, clover_inv, (cudaStream_t)stream);
    return run_clover_build(make_geo(g), g->prec, 4.0 + m0, csw, expo, u_fund, clover_fwd, clover_inv, (cudaStream_t)stream);
}

int hr_clover_build(const hr_geom* g, double m0, double csw, const void* u_fund, void* clover_fwd,
                    void* clover_inv, void* stream) {
    return clover_build_any(g, m0, csw, 0, u_fund, clover_fwd, clover_inv, stream);
}

int hr_clover_build_exp(const hr_geom* g, double m0, double csw, const void* u_fund, void* clover_fwd,
                        void* clover_inv, void* stream) {
    return clover_build_any(g, m0, csw, 1, u_fund, clover_fwd, clover_inv, stream);
}

int hr_clover_apply(const hr_geom* g, int parity, const void* blocks, const void* in, void* out, void* stream) {
    HR_TRY(check_geom(g));
    if (parity < HR_EVEN || parity > HR_BOTH) { set_error("hr_clover_apply: parity %d", parity); return HR_EINVAL; }
    HR_TRY(check_ptr(blocks, "blocks")); HR_TRY(check_ptr(in, "in")); HR_TRY(check_ptr(out, "out"));
    return run_clover_apply(make_geo(g), g->rep, g->prec, parity, blocks, in, out, (cudaStream_t)stream);
}

int hr_clover_count_nonfinite(const hr_geom* g, const void* blocks, void* count_dev, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_ptr(blocks, "blocks"));
    if (!count_dev || (reinterpret_cast<uintptr_t>(count_dev) & 7)) { set_error("hr_clover_count_nonfinite: count_dev must be an 8-byte aligned device pointer"); return HR_EINVAL; }
    return run_count_nonfinite(g->prec, blocks, hr_clover_bytes(g), reinterpret_cast<unsigned long long*>(count_dev), (cudaStream_t)stream);
}

// ---------------------------------------------------------------- S1
size_t hr_cg_workspace_bytes(const hr_geom* g) {
    if (!geom_ok(g)) return 0;
    return cg_workspace_bytes(g);
}

int hr_cg_solve(const hr_geom* g, double m0, const void* u, const void* clover_fwd, const void* clover_inv,
                const void* b, void* x, void* workspace, double tol, int max_iter, int check_every,
                int* iters, double* relres, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_links(g));
    HR_TRY(check_ptr(u, "u")); HR_TRY(check_ptr(b, "b")); HR_TRY(check_ptr(x, "x")); HR_TRY(check_ptr(workspace, "workspace"));
    if (!(tol > 0.0) || max_iter < 0 || check_every < 1) { set_error("hr_cg_solve: tol must be > 0, max_iter >= 0, check_every >= 1"); return HR_EINVAL; }
    if ((clover_fwd == nullptr) != (clover_inv == nullptr)) { set_error("hr_cg_solve: clover_fwd and clover_inv must both be given"); return HR_EINVAL; }
    const size_t half = half_spinor_bytes(g);
    if (overlap(b, half, x, half)) { set_error("hr_cg_solve: x aliases b"); return HR_EINVAL; }
    if (overlap(workspace, cg_workspace_bytes(g), x, half) || overlap(workspace, cg_workspace_bytes(g), b, half)) {
        set_error("hr_cg_solve: workspace aliases b or x");
        return HR_EINVAL;
    }
    return run_cg(g, m0, u, clover_fwd, clover_inv, b, x, workspace, tol, max_iter, check_every, iters, relres, (cudaStream_t)stream);
}

size_t hr_cg_mixed_workspace_bytes(const hr_geom* g) {
    if (!geom_ok(g) || g->prec != HR_PREC_F64) return 0;
    return cg_mixed_workspace_bytes(g);
}

static int cg_mixed_any(const hr_geom* g, double m0, const void* u_f64, const void* u_f32, const void* cf64, const void* ci64,
                        const void* cf32, const void* ci32, const void* b, void* x, void* workspace,
                        double tol, double inner_tol, int max_outer, int max_inner, int check_every,
                        int* outer_iters, int* inner_iters, double* relres, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_links(g));
    if (g->prec != HR_PREC_F64) { set_error("hr_cg_solve_mixed: the geometry describes the fp64 fields (prec must be HR_PREC_F64)"); return HR_EINVAL; }
    HR_TRY(check_ptr(u_f64, "u_f64")); HR_TRY(check_ptr(u_f32, "u_f32")); HR_TRY(check_ptr(b, "b")); HR_TRY(check_ptr(x, "x"));
    HR_TRY(check_ptr(workspace, "workspace"));
    const int nclover = (cf64 != nullptr) + (ci64 != nullptr) + (cf32 != nullptr) + (ci32 != nullptr);
    if (nclover != 0 && nclover != 4) { set_error("hr_cg_solve_mixed_clover: the four clover block fields must all be given"); return HR_EINVAL; }
    if (!(tol > 0.0) || !(inner_tol > 0.0) || inner_tol >= 1.0 || max_outer < 0 || max_inner < 1 || check_every < 1) {
        set_error("hr_cg_solve_mixed: need tol > 0, 0 < inner_tol < 1, max_outer >= 0, max_inner >= 1, check_every >= 1");
        return HR_EINVAL;
    }
    const size_t half = half_spinor_bytes(g);
    if (overlap(b, half, x, half) || overlap(workspace, cg_mixed_workspace_bytes(g), x, half) || overlap(workspace, cg_mixed_workspace_bytes(g), b, half)) {
        set_error("hr_cg_solve_mixed: b, x and workspace must not overlap");
        return HR_EINVAL;
    }
    return run_cg_mixed(g, m0, u_f64, u_f32, cf64, ci64, cf32, ci32, b, x, workspace, tol, inner_tol, max_outer, max_inner, check_every,
                        outer_iters, inner_iters, relres, (cudaStream_t)stream);
}

int hr_cg_solve_mixed(const hr_geom* g, double m0, const void* u_f64, const void* u_f32, const void* b, void* x, void* workspace,
                      double tol, double inner_tol, int max_outer, int max_inner, int check_every,
                      int* outer_iters, int* inner_iters, double* relres, void* stream) {
    return cg_mixed_any(g, m0, u_f64, u_f32, nullptr, nullptr, nullptr, nullptr, b, x, workspace, tol, inner_tol, max_outer, max_inner,
                        check_every, outer_iters, inner_iters, relres, stream);
}

int hr_cg_solve_mixed_clover(const hr_geom* g, double m0, const void* u_f64, const void* u_f32,
                             const void* clover_fwd_f64, const void* clover_inv_f64, const void* clover_fwd_f32, const void* clover_inv_f32,
                             const void* b, void* x, void* workspace, double tol, double inner_tol, int max_outer, int max_inner,
                             int check_every, int* outer_iters, int* inner_iters, double* relres, void* stream) {
    return cg_mixed_any(g, m0, u_f64, u_f32, clover_fwd_f64, clover_inv_f64, clover_fwd_f32, clover_inv_f32, b, x, workspace, tol, inner_tol,
                        max_outer, max_inner, check_every, outer_iters, inner_iters, relres, stream);
}

// ---------------------------------------------------------------- M1
int hr_dirac_flops_bytes(const hr_geom* g, int op, double* flops_per_site, double* bytes_compulsory,
                         double* bytes_requested) {
    HR_TRY(check_geom(g));
    const double N = ncolour(g->rep), w = (double)real_bytes(g->prec);
    const double nr = 8.0 * N, S = nr * w;
    const double Gf = (g->link_storage != HR_LINKS_FULL ? 4.0 : 8.0) * w, Ga = 9.0 * w;
    const double G = g->rep == HR_REP_FUND ? Gf : g->rep == HR_REP_SU3 ? (g->link_storage == HR_LINKS_COMPRESSED ? 12.0 : 18.0) * w : (g->link_storage == HR_LINKS_ONTHEFLY ? 4.0 * w : Ga);
    const double Bk = 2.0 * (2 * N) * (2 * N) * w;            // two hermitian 2N x 2N blocks per site
    // per direction: 4N adds to project, two colour mat-vecs, 8N adds to accumulate; x8, minus the first accumulate
    // (rebuilding R from the quaternion, ~30 flops per link, is not counted: the model counts the operator's flops)
    const double Fhop = g->rep != HR_REP_ADJ ? 8.0 * N * (16.0 * N + 7.0) : 8.0 * N * (8.0 * N + 7.0);   // complex links (624, SU(3): 1320) : real links (744)
    const double Fblk = 2.0 * (2.0 * (2 * N) + 8.0 * (2 * N) * (2 * N - 1));   // two hermitian 2N x 2N mat-vecs: 208 (fund), 504 (adj)
    double f = 0, bc = 0, br = 0;
    if (g->rep == HR_REP_SU3 && op == HR_OP_REPRESENT) return check_no_su3(g, "hr_dirac_flops_bytes of the representation op");
    switch (op) {
        case HR_OP_HOP: f = Fhop; bc = 2 * S + 8 * G; br = 9 * S + 8 * G; break;
        case HR_OP_DIRAC: f = Fhop + 3 * nr; bc = 2 * S + 4 * G; br = 10 * S + 8 * G; break;
        case HR_OP_DHAT: f = 2 * Fhop + 3 * nr; bc = 5 * S + 16 * G; br = 19 * S + 16 * G; break;
        case HR_OP_CLOVER:
            f = Fblk; bc = 2 * S + Bk; br = bc; break;
        case HR_OP_DHAT_CLOVER:
            f = 2 * Fhop + 2 * Fblk + 2 * nr; bc = 5 * S + 16 * G + 2 * Bk; br = 19 * S + 16 * G + 2 * Bk; break;
        case HR_OP_REPRESENT: f = 4 * 30.0; bc = 4 * Gf + 4 * Ga; br = bc; break;
        default: set_error("hr_dirac_flops_bytes: unknown op %d", op); return HR_EINVAL;
    }
    if (flops_per_site) *flops_per_site = f;
    if (bytes_compulsory) *bytes_compulsory = bc;
    if (bytes_requested) *bytes_requested = br;
    return HR_OK;
}

// ---------------------------------------------------------------- host-buffer path
static size_t up256(size_t n) { return (n + 255) & ~(size_t)255; }

size_t hr_host_workspace_bytes(const hr_geom* g) {
    if (!geom_ok(g)) return 0;
    const int urep = g->link_storage == HR_LINKS_ONTHEFLY ? HR_REP_FUND : g->rep;   // representation of the links handed in
    return up256(hr_canonical_gauge_bytes(g, urep)) + 2 * up256(hr_canonical_spinor_bytes(g)) +
           up256(hr_gauge_bytes(g, urep)) + 3 * up256(hr_spinor_bytes(g, HR_BOTH));
}

static int host_apply(const hr_geom* g, int op, double m0, const void* u_h, const void* in_h, void* out_h,
                      void* workspace, void* stream) {
    HR_TRY(check_geom(g)); HR_TRY(check_links(g));
    if (!u_h || !in_h || !out_h) { set_error("host pointer is NULL"); return HR_EINVAL; }
    HR_TRY(check_ptr(workspace, "workspace"));
    cudaStream_t st = (cudaStream_t)stream;
    const int urep = g->link_storage == HR_LINKS_ONTHEFLY ? HR_REP_FUND : g->rep;
    const size_t cg = hr_canonical_gauge_bytes(g, urep), cs = hr_canonical_spinor_bytes(g);
    const size_t dg = hr_gauge_bytes(g, urep), ds = hr_spinor_bytes(g, HR_BOTH), half = ds / 2;
    char* w = (char*)workspace;
    char* c_u = w; w += up256(cg);
    char* c_in = w; w += up256(cs);
    char* c_out = w; w += up256(cs);
    char* d_u = w; w += up256(dg);
    char* d_in = w; w += up256(ds);
    char* d_out = w; w += up256(ds);
    char* d_tmp = w;
#define HR_CUDA(call)                                                         \
    do {                                                                      \
        cudaError_t e_ = (call);                                              \
        if (e_ != cudaSuccess) { set_error("%s: %s", #call, cudaGetErrorString(e_)); return HR_ECUDA; } \
    } while (0)
    HR_CUDA(cudaMemcpyAsync(c_u, u_h, cg, cudaMemcpyHostToDevice, st));
    HR_CUDA(cudaMemcpyAsync(c_in, in_h, cs, cudaMemcpyHostToDevice, st));
    HR_TRY(hr_pack_gauge(g, urep, c_u, d_u, stream));
    HR_TRY(hr_pack_spinor(g, c_in, d_in, stream));
    if (op < 0) {
        HR_TRY(hr_dirac_apply(g, m0, d_u, d_in, d_out, stream));
    } else {
        // outputs of the untouched parity come back as zeros
        HR_CUDA(cudaMemsetAsync(d_out, 0, ds, st));
        const int in_par = (op == HR_EO_HOP_EO) ? HR_ODD : HR_EVEN;
        const int out_par = (op == HR_EO_HOP_OE) ? HR_ODD : HR_EVEN;
        HR_TRY(hr_dirac_eo_apply(g, op, m0, d_u, nullptr, nullptr, d_in + in_par * half, d_out + out_par * half, d_tmp, stream));
    }
    HR_TRY(hr_unpack_spinor(g, d_out, c_out, stream));
    HR_CUDA(cudaMemcpyAsync(out_h, c_out, cs, cudaMemcpyDeviceToHost, st));
    HR_CUDA(cudaStreamSynchronize(st));
#undef HR_CUDA
    return HR_OK;
}

int hr_dirac_apply_host(const hr_geom* g, double m0, const void* u_canon_host, const void* psi_canon_host,
                        void* out_canon_host, void* workspace, void* stream) {
    return host_apply(g, -1, m0, u_canon_host, psi_canon_host, out_canon_host, workspace, stream);
}

int hr_dirac_eo_apply_host(const hr_geom* g, int op, double m0, const void* u_canon_host,
                           const void* in_canon_host, void* out_canon_host, void* workspace, void* stream) {
    if (op < HR_EO_HOP_OE || op > HR_EO_DHAT) { set_error("hr_dirac_eo_apply_host: unknown op %d", op); return HR_EINVAL; }
    return host_apply(g, op, m0, u_canon_host, in_canon_host, out_canon_host, workspace, stream);
}

// ---------------------------------------------------------------- diagnostics
size_t hr_last_error(char* buf, size_t len) {
    const size_t n = strlen(g_err);
    if (buf && len) {
        const size_t m = n < len - 1 ? n : len - 1;
        memcpy(buf, g_err, m);
        buf[m] = 0;
    }
    return n;
}

unsigned long long hr_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

int hr_kernel_plan(const hr_geom* g, int op, int* info) {
    HR_TRY(check_geom(g));
    if (!info) { set_error("hr_kernel_plan: info is NULL"); return HR_EINVAL; }
    if (op != HR_OP_HOP && op != HR_OP_DIRAC) { set_error("hr_kernel_plan: op must be HR_OP_HOP or HR_OP_DIRAC"); return HR_EINVAL; }
    return kernel_plan(g, op == HR_OP_DIRAC ? 2 : 0, info);
}

const char* hr_kernel_name(const hr_geom* g) {
    if (!geom_ok(g)) return "invalid";
    return tiled_chosen(g) ? "tiled" : "generic";
}

}  // extern "C"
