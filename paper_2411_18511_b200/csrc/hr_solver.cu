// hr_solver.cu — conjugate gradient on the normal equations of the even-odd operator (
// PAPER.md:13 "range of inverters", PAPER.md:39 the even-odd operator "used mainly in the HMC"):
//     Dhat^dag Dhat x = b   on the even sites,   Dhat^dag = gamma5 Dhat gamma5.
// The operator applications are the hopping kernels; the linear algebra between them rides in the epilogue of the second hop
// of each Dhat (POST_G5_NORM, POST_CG_UPDATE of hr_hop_generic.cuh: s = gamma5 Dhat p with |Dhat p|^2, and r -= alpha gamma5 Dhat s
// with |r|^2), so Dhat p and Dhat s never reach memory; x += alpha p and p = r + beta p share the one vector kernel left.  Every scalar
// stays on the device, so an iteration is enqueued without a host round trip.  Reductions are two-stage with a fixed order (one
// partial sum per CTA in double, then one block sums them): results are bitwise reproducible from run to run.
#include "hr_hop_generic.cuh"

namespace hr {

constexpr int CG_BLOCK = 256;
constexpr int CG_MAX_PARTIALS = 148 * 8;

// device scalars of the iteration
struct CgScalars {
    double rr;      // <r,r>
    double rr_new;
    double pap;     // <p, Dhat^dag Dhat p> = |Dhat p|^2
    double bb;      // <b,b>
    double alpha, beta;
};

// sign of gamma5 = diag(1,1,-1,-1) on 16-byte chunk number `chunk` of a half field laid out [row][NCH][L3h]
__device__ __forceinline__ double g5_sign(size_t chunk, int L3h, int NCH) {
    const int c = (int)((chunk / (size_t)L3h) % (size_t)NCH);
    return c < NCH / 2 ? 1.0 : -1.0;
}

template <typename T> struct RealsPerChunk { static constexpr int value = 16 / sizeof(T); };

__device__ __forceinline__ double block_sum(double v) {
    __shared__ double sm[CG_BLOCK / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int i = 0; i < CG_BLOCK / 32; ++i) t += sm[i];
    return t;   // valid in thread 0
}

// s = gamma5 t, partial[blockIdx] = sum |t|^2            (t = Dhat p;  |t|^2 = <p, Dhat^dag Dhat p>)
template <typename T>
__global__ void __launch_bounds__(CG_BLOCK) cg_g5_norm_kernel(size_t nchunks, int L3h, int NCH, const void* __restrict__ t_, void* __restrict__ s_,
                                                              double* __restrict__ partial) {
    typedef typename Chunk<T>::type chunk_t;
    constexpr int R = RealsPerChunk<T>::value;
    const chunk_t* t = reinterpret_cast<const chunk_t*>(t_);
    chunk_t* s = reinterpret_cast<chunk_t*>(s_);
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nchunks; i += (size_t)gridDim.x * blockDim.x) {
        T e[R];
        chunk_to_reals(ldg16<LD_STREAM>(t + i), e);
        const T sg = (T)g5_sign(i, L3h, NCH);
#pragma unroll
        for (int k = 0; k < R; ++k) {
            acc += (double)e[k] * (double)e[k];
            e[k] *= sg;
        }
        s[i] = reals_to_chunk(e);
    }
    const double tot = block_sum(acc);
    if (threadIdx.x == 0) partial[blockIdx.x] = tot;
}

// which scalar a finalize step produces
enum { CG_FIN_INIT = 0, CG_FIN_PAP = 1, CG_FIN_RR = 2 };

// one block: sums the partials in index order and updates the scalars
__global__ void __launch_bounds__(CG_BLOCK) cg_finalize_kernel(int what, int npartial, const double* __restrict__ partial, CgScalars* sc) {
    __shared__ double sm[CG_BLOCK];
    double v = 0.0;
    for (int i = threadIdx.x; i < npartial; i += CG_BLOCK) v += partial[i];
    sm[threadIdx.x] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int i = 0; i < CG_BLOCK; ++i) t += sm[i];
        if (what == CG_FIN_INIT) {
            sc->rr = t; sc->bb = t; sc->rr_new = t; sc->alpha = 0.0; sc->beta = 0.0; sc->pap = 0.0;
        } else if (what == CG_FIN_PAP) {
            sc->pap = t;
            sc->alpha = t > 0.0 ? sc->rr / t : 0.0;
        } else {
            sc->rr_new = t;
            sc->beta = sc->rr > 0.0 ? t / sc->rr : 0.0;
            sc->rr = t;
        }
    }
}

// x += alpha p;  p = r + beta p        (alpha, beta of this iteration; r already updated by the POST_CG_UPDATE hop)
template <typename T>
__global__ void __launch_bounds__(CG_BLOCK) cg_direction_kernel(size_t nchunks, const CgScalars* __restrict__ sc, const void* __restrict__ r_, void* __restrict__ p_,
                                                                void* __restrict__ x_) {
    typedef typename Chunk<T>::type chunk_t;
    constexpr int R = RealsPerChunk<T>::value;
    const chunk_t* r = reinterpret_cast<const chunk_t*>(r_);
    chunk_t* p = reinterpret_cast<chunk_t*>(p_);
    chunk_t* x = reinterpret_cast<chunk_t*>(x_);
    const T alpha = (T)sc->alpha, beta = (T)sc->beta;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nchunks; i += (size_t)gridDim.x * blockDim.x) {
        T er[R], ep[R], ex[R];
        chunk_to_reals(ldg16<LD_STREAM>(r + i), er);
        chunk_to_reals(p[i], ep);
        chunk_to_reals(x[i], ex);
#pragma unroll
        for (int k = 0; k < R; ++k) {
            ex[k] = fma(alpha, ep[k], ex[k]);
            ep[k] = fma(beta, ep[k], er[k]);
        }
        x[i] = reals_to_chunk(ex);
        p[i] = reals_to_chunk(ep);
    }
}

// r = b, p = b, x = 0, partial = sum |b|^2
template <typename T>
__global__ void __launch_bounds__(CG_BLOCK) cg_init_kernel(size_t nchunks, const void* __restrict__ b_, void* __restrict__ x_, void* __restrict__ r_,
                                                           void* __restrict__ p_, double* __restrict__ partial) {
    typedef typename Chunk<T>::type chunk_t;
    constexpr int R = RealsPerChunk<T>::value;
    const chunk_t* b = reinterpret_cast<const chunk_t*>(b_);
    chunk_t* x = reinterpret_cast<chunk_t*>(x_);
    chunk_t* r = reinterpret_cast<chunk_t*>(r_);
    chunk_t* p = reinterpret_cast<chunk_t*>(p_);
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nchunks; i += (size_t)gridDim.x * blockDim.x) {
        T e[R], z[R];
        const chunk_t v = b[i];
        chunk_to_reals(v, e);
#pragma unroll
        for (int k = 0; k < R; ++k) { acc += (double)e[k] * (double)e[k]; z[k] = (T)0; }
        r[i] = v;
        p[i] = v;
        x[i] = reals_to_chunk(z);
    }
    const double tot = block_sum(acc);
    if (threadIdx.x == 0) partial[blockIdx.x] = tot;
}

// ------------------------------------------------------------------ host driver
static size_t up256s(size_t n) { return (n + 255) & ~(size_t)255; }

// partial sums: one per block of the vector kernels (<= CG_MAX_PARTIALS) or per CTA of a hop that carries a CG stage
static size_t cg_partials(const hr_geom* g) {
    const size_t nb = (size_t)hop_post_blocks(g);
    return nb > (size_t)CG_MAX_PARTIALS ? nb : (size_t)CG_MAX_PARTIALS;
}

size_t cg_workspace_bytes(const hr_geom* g) {
    const size_t half = hr_spinor_bytes(g, HR_EVEN);
    return 256 + up256s(cg_partials(g) * sizeof(double)) + 5 * up256s(half);
}

template <typename T>
static int cg_run(const hr_geom* g, double m0, const void* u, const void* cf, const void* ci, const void* b, void* x, void* workspace,
                  double tol, int max_iter, int check_every, int* iters_out, double* relres_out, cudaStream_t st) {
    const Geo geo = make_geo(g);
    const int NCH = spinor_chunks(g->rep, g->prec);
    const size_t half = hr_spinor_bytes(g, HR_EVEN);
    const size_t nchunks = half / 16;
    char* w8 = (char*)workspace;
    CgScalars* sc = (CgScalars*)w8; w8 += 256;
    double* partial = (double*)w8; w8 += up256s(cg_partials(g) * sizeof(double));
    void* r = w8; w8 += up256s(half);
    void* p = w8; w8 += up256s(half);
    w8 += up256s(half);      // (a third vector of the unfused iteration: kept in the layout, unused)
    void* w = w8; w8 += up256s(half);
    void* tmp = w8;
    int nblk = (int)((nchunks + CG_BLOCK - 1) / CG_BLOCK);
    if (nblk > CG_MAX_PARTIALS) nblk = CG_MAX_PARTIALS;
    const bool clover = cf && ci;
    const double d = 4.0 + m0;
    if (!clover && d == 0.0) { set_error("hr_cg_solve: 4+m0 = 0, D_oo is singular"); return HR_EINVAL; }
    const int nhop = hop_post_blocks(g);

    cg_init_kernel<T><<<nblk, CG_BLOCK, 0, st>>>(nchunks, b, x, r, p, partial);
    cg_finalize_kernel<<<1, CG_BLOCK, 0, st>>>(CG_FIN_INIT, nblk, partial, sc);
    count_launch(2);
    int rc = check_launch("cg_init_kernel");
    if (rc != HR_OK) return rc;

    CgScalars h;
    int it = 0;
    double relres = 1.0;
    bool done = false;
    while (!done) {
        // convergence is read back every check_every iterations (the only host round trip of the solve)
        if (it % check_every == 0 || it >= max_iter) {
            cudaError_t e = cudaMemcpyAsync(&h, sc, sizeof(h), cudaMemcpyDeviceToHost, st);
            if (e == cudaSuccess) e = cudaStreamSynchronize(st);
            if (e != cudaSuccess) { set_error("hr_cg_solve: %s", cudaGetErrorString(e)); return HR_ECUDA; }
            if (!(h.rr == h.rr) || !(h.bb == h.bb)) { set_error("hr_cg_solve: residual is NaN at iteration %d", it); return HR_ECUDA; }
            relres = h.bb > 0.0 ? sqrt(h.rr / h.bb) : 0.0;
            if (h.bb == 0.0 || h.rr <= tol * tol * h.bb || it >= max_iter) { done = true; break; }
        }
        // One iteration = four hops and one vector kernel.  The linear algebra between the operator applications rides in the
        // epilogues of the second hop of each Dhat (hr_hop_generic.cuh: POST_*), so Dhat p and Dhat s are never written out:
        //   tmp = [A_oo^-1] H_oe p ;  s = gamma5 (Dhat p) with <p, Dhat^dag Dhat p> = |Dhat p|^2 as per-CTA partial sums      (POST_G5_NORM)
        //   tmp = [A_oo^-1] H_oe s ;  r -= alpha gamma5 (Dhat s), |r|^2                                                     (POST_CG_UPDATE)
        //   x += alpha p ;  p = r + beta p
        HopArgs a;
        a.gauge = u; a.both = 0; a.partial = partial;
        a.in = p; a.out = tmp; a.parity = HR_ODD; a.phi = nullptr; a.clover = clover ? ci : nullptr; a.a = 0.0; a.c = 1.0;
        rc = run_hop(g, a, clover ? EPI_CLOVER_INV : EPI_NONE, st);
        if (rc != HR_OK) return rc;
        a.in = tmp; a.out = w; a.parity = HR_EVEN; a.phi = p; a.clover = clover ? cf : nullptr; a.a = clover ? 0.0 : d; a.c = clover ? -0.25 : -1.0 / (4.0 * d);
        rc = run_hop_post(g, a, clover ? EPI_CLOVER_AXPY : EPI_AXPY, POST_G5_NORM, st);
        if (rc != HR_OK) return rc;
        cg_finalize_kernel<<<1, CG_BLOCK, 0, st>>>(CG_FIN_PAP, nhop, partial, sc);
        a.in = w; a.out = tmp; a.parity = HR_ODD; a.phi = nullptr; a.clover = clover ? ci : nullptr; a.a = 0.0; a.c = 1.0;
        rc = run_hop(g, a, clover ? EPI_CLOVER_INV : EPI_NONE, st);
        if (rc != HR_OK) return rc;
        a.in = tmp; a.out = nullptr; a.parity = HR_EVEN; a.phi = w; a.clover = clover ? cf : nullptr; a.a = clover ? 0.0 : d; a.c = clover ? -0.25 : -1.0 / (4.0 * d);
        a.cg_alpha = &sc->alpha; a.cg_r = r;
        rc = run_hop_post(g, a, clover ? EPI_CLOVER_AXPY : EPI_AXPY, POST_CG_UPDATE, st);
        if (rc != HR_OK) return rc;
        cg_finalize_kernel<<<1, CG_BLOCK, 0, st>>>(CG_FIN_RR, nhop, partial, sc);
        cg_direction_kernel<T><<<nblk, CG_BLOCK, 0, st>>>(nchunks, sc, r, p, x);
        count_launch(3);
        rc = check_launch("cg iteration");
        if (rc != HR_OK) return rc;
        ++it;
    }
    if (iters_out) *iters_out = it;
    if (relres_out) *relres_out = relres;
    return HR_OK;
}

int run_cg(const hr_geom* g, double m0, const void* u, const void* cf, const void* ci, const void* b, void* x, void* workspace, double tol,
           int max_iter, int check_every, int* iters_out, double* relres_out, cudaStream_t st) {
    if (g->prec == HR_PREC_F64) return cg_run<double>(g, m0, u, cf, ci, b, x, workspace, tol, max_iter, check_every, iters_out, relres_out, st);
    return cg_run<float>(g, m0, u, cf, ci, b, x, workspace, tol, max_iter, check_every, iters_out, relres_out, st);
}

// ------------------------------------------------------------------ mixed precision: fp64 defect correction around fp32 CG
// (SURVEY.md §8(f) item 2 "mixed fp32/fp64 defect correction").  Outer loop in double:
//     r = b - Dhat^dag Dhat x  (true residual, fp64 operator);  stop when |r| <= tol |b|;
//     solve Dhat^dag Dhat e = r in fp32 to the relative accuracy inner_tol (cg_run<float>);  x += e.
// The fp32 fields use their own device layout (two complex per 16-byte chunk), so r and e are converted site by site.

// one thread per fp32 chunk: complex numbers 2c, 2c+1 of site (row, h):  f64 chunks (row*NC + 2c [+1])*L3h + h
__global__ void __launch_bounds__(CG_BLOCK) cg_to_f32_kernel(size_t nchunks32, int L3h, int NCH32, const double2* __restrict__ src, float4* __restrict__ dst) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nchunks32; i += (size_t)gridDim.x * blockDim.x) {
        const size_t h = i % L3h, rc = i / L3h;          // rc = row*NCH32 + c
        const size_t row = rc / NCH32, c = rc % NCH32;
        const size_t j = (row * (2 * NCH32) + 2 * c) * L3h + h;
        const double2 a = src[j], b = src[j + L3h];
        dst[i] = make_float4((float)a.x, (float)a.y, (float)b.x, (float)b.y);
    }
}
// x += e (e in fp32 layout)
__global__ void __launch_bounds__(CG_BLOCK) cg_add_f32_kernel(size_t nchunks32, int L3h, int NCH32, const float4* __restrict__ e, double2* __restrict__ x) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nchunks32; i += (size_t)gridDim.x * blockDim.x) {
        const size_t h = i % L3h, rc = i / L3h;
        const size_t row = rc / NCH32, c = rc % NCH32;
        const size_t j = (row * (2 * NCH32) + 2 * c) * L3h + h;
        const float4 v = e[i];
        double2 a = x[j], b = x[j + L3h];
        a.x += (double)v.x; a.y += (double)v.y; b.x += (double)v.z; b.y += (double)v.w;
        x[j] = a;
        x[j + L3h] = b;
    }
}
// r = b - gamma5 w, partial = sum |r|^2      (w = Dhat gamma5 Dhat x)
__global__ void __launch_bounds__(CG_BLOCK) cg_residual_kernel(size_t nchunks, int L3h, int NCH, const double2* __restrict__ b, const double2* __restrict__ w,
                                                               double2* __restrict__ r, double* __restrict__ partial) {
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nchunks; i += (size_t)gridDim.x * blockDim.x) {
        const double sg = g5_sign(i, L3h, NCH);
        const double2 bv = b[i], wv = w[i];
        double2 rv;
        rv.x = bv.x - sg * wv.x;
        rv.y = bv.y - sg * wv.y;
        acc += rv.x * rv.x + rv.y * rv.y;
        r[i] = rv;
    }
    const double tot = block_sum(acc);
    if (threadIdx.x == 0) partial[blockIdx.x] = tot;
}
__global__ void __launch_bounds__(CG_BLOCK) cg_zero_kernel(size_t nchunks, double2* __restrict__ x) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nchunks; i += (size_t)gridDim.x * blockDim.x) x[i] = make_double2(0.0, 0.0);
}

static hr_geom as_f32(const hr_geom* g) {
    hr_geom g32 = *g;
    g32.prec = HR_PREC_F32;
    return g32;
}

size_t cg_mixed_workspace_bytes(const hr_geom* g) {
    const hr_geom g32 = as_f32(g);
    const size_t half64 = hr_spinor_bytes(g, HR_EVEN), half32 = hr_spinor_bytes(&g32, HR_EVEN);
    return 256 + up256s(CG_MAX_PARTIALS * sizeof(double)) + 4 * up256s(half64) + 2 * up256s(half32) + up256s(cg_workspace_bytes(&g32));
}

int run_cg_mixed(const hr_geom* g, double m0, const void* u64, const void* u32, const void* cf64, const void* ci64, const void* cf32, const void* ci32,
                 const void* b, void* x, void* workspace, double tol, double inner_tol,
                 int max_outer, int max_inner, int check_every, int* outer_out, int* inner_out, double* relres_out, cudaStream_t st) {
    const hr_geom g32 = as_f32(g);
    const Geo geo = make_geo(g);
    const int NCH = spinor_chunks(g->rep, g->prec), NCH32 = spinor_chunks(g->rep, HR_PREC_F32);
    const size_t half64 = hr_spinor_bytes(g, HR_EVEN), half32 = hr_spinor_bytes(&g32, HR_EVEN);
    const size_t nchunks = half64 / 16, nchunks32 = half32 / 16;
    char* w8 = (char*)workspace;
    CgScalars* sc = (CgScalars*)w8; w8 += 256;
    double* partial = (double*)w8; w8 += up256s(CG_MAX_PARTIALS * sizeof(double));
    void* r = w8; w8 += up256s(half64);
    void* t = w8; w8 += up256s(half64);
    void* w = w8; w8 += up256s(half64);
    void* tmp = w8; w8 += up256s(half64);
    void* r32 = w8; w8 += up256s(half32);
    void* e32 = w8; w8 += up256s(half32);
    void* ws32 = w8;
    int nblk = (int)((nchunks + CG_BLOCK - 1) / CG_BLOCK);
    if (nblk > CG_MAX_PARTIALS) nblk = CG_MAX_PARTIALS;
    int nblk32 = (int)((nchunks32 + CG_BLOCK - 1) / CG_BLOCK);
    if (nblk32 > CG_MAX_PARTIALS) nblk32 = CG_MAX_PARTIALS;
    void* strm = (void*)st;

    cg_zero_kernel<<<nblk, CG_BLOCK, 0, st>>>(nchunks, (double2*)x);
    count_launch();
    double bb = -1.0, relres = 1.0;
    int outer = 0, inner_total = 0;
    for (;;) {
        // r = b - Dhat^dag Dhat x in double; on the first pass x = 0, so r = b and |b|^2 come from the residual kernel
        // alone (with w = x = 0) and the two fp64 operator applications are skipped
        int rc = HR_OK;
        if (bb < 0.0) {
            cg_residual_kernel<<<nblk, CG_BLOCK, 0, st>>>(nchunks, geo.L3h, NCH, (const double2*)b, (const double2*)x, (double2*)r, partial);
            count_launch();
        } else {
            rc = hr_dirac_eo_apply(g, HR_EO_DHAT, m0, u64, cf64, ci64, x, t, tmp, strm);
            if (rc != HR_OK) return rc;
            cg_g5_norm_kernel<double><<<nblk, CG_BLOCK, 0, st>>>(nchunks, geo.L3h, NCH, t, w, partial);
            rc = hr_dirac_eo_apply(g, HR_EO_DHAT, m0, u64, cf64, ci64, w, t, tmp, strm);
            if (rc != HR_OK) return rc;
            cg_residual_kernel<<<nblk, CG_BLOCK, 0, st>>>(nchunks, geo.L3h, NCH, (const double2*)b, (const double2*)t, (double2*)r, partial);
            count_launch(2);
        }
        cg_finalize_kernel<<<1, CG_BLOCK, 0, st>>>(CG_FIN_INIT, nblk, partial, sc);
        count_launch();
        CgScalars h;
        cudaError_t e = cudaMemcpyAsync(&h, sc, sizeof(h), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { set_error("hr_cg_solve_mixed: %s", cudaGetErrorString(e)); return HR_ECUDA; }
        if (!(h.rr == h.rr)) { set_error("hr_cg_solve_mixed: residual is NaN after %d outer iterations", outer); return HR_ECUDA; }
        if (bb < 0.0) bb = h.rr;                         // first pass: x = 0, so |r|^2 = |b|^2
        relres = bb > 0.0 ? sqrt(h.rr / bb) : 0.0;
        if (bb == 0.0 || relres <= tol || outer >= max_outer) break;
        // inner solve in fp32: Dhat^dag Dhat e = r
        cg_to_f32_kernel<<<nblk32, CG_BLOCK, 0, st>>>(nchunks32, geo.L3h, NCH32, (const double2*)r, (float4*)r32);
        count_launch();
        int it = 0;
        double rel32 = 0.0;
        rc = run_cg(&g32, m0, u32, cf32, ci32, r32, e32, ws32, inner_tol, max_inner, check_every, &it, &rel32, st);
        if (rc != HR_OK) return rc;
        inner_total += it;
        cg_add_f32_kernel<<<nblk32, CG_BLOCK, 0, st>>>(nchunks32, geo.L3h, NCH32, (const float4*)e32, (double2*)x);
        count_launch();
        rc = check_launch("cg mixed outer iteration");
        if (rc != HR_OK) return rc;
        ++outer;
    }
    if (outer_out) *outer_out = outer;
    if (inner_out) *inner_out = inner_total;
    if (relres_out) *relres_out = relres;
    return HR_OK;
}

}  // namespace hr
