/* hr_dslash.h — C-ABI of the B200-native Wilson-Dirac hot path of HiRep (arXiv 2411.18511).
 *
 * What the paper describes (§2.1 "Wilson-Dirac Operator", §2.2 "Clover
 * improvement") is a set of device kernels; it prints no formula.  The operator is the one written in
 * BASELINE.json `north_star`,
 *
 *     D psi(x) = (4+m0) psi(x) - 1/2 sum_mu [ (1-gamma_mu) U_mu(x) psi(x+mu) + (1+gamma_mu) U_mu(x-mu)^dag psi(x-mu) ],
 *
 * on a 4-D periodic lattice, gauge group SU(2), fermions in the fundamental (2 complex colours) or
 * adjoint (3 colours, real 3x3 links) representation, with the conventions of SURVEY.md §8(c) /
 * DESIGN.md §3 (gamma basis A2, site order A3, canonical formats A4).
 *
 * Conventions of every call
 *   - extern "C", plain C types, no torch types.  `stream` is a cudaStream_t passed as void* (NULL = default).
 *   - Unless the name ends in `_host`, every data pointer is a DEVICE pointer, 16-byte aligned.
 *   - Return value: HR_OK, or an error code below; hr_last_error() gives the text of the last failure
 *     of the calling thread.  Argument checks happen before anything is enqueued.
 *   - Device calls only enqueue work on `stream`: no allocation, no host-device synchronisation.
 *   - The caller owns every buffer, including temporaries, and sizes them with the hr_*_bytes queries.
 *   - "canonical" = array-of-structs in lexicographic site order (x3 fastest), real type of geom->prec:
 *         spinor        [V][4 spin][N colour][re,im]
 *         fund gauge    [V][4 mu][2 row][2 col][re,im]
 *         adj gauge     [V][4 mu][3 a][3 b]                       (real)
 *         SU(3) gauge   [V][4 mu][3 row][3 col][re,im]            (HR_REP_SU3)
 *         clover blocks [V][2 chirality +,-][(2N)^2 reals]        one hermitian 2N x 2N block per chirality, N = 2 / 3
 *                        colours: 2N real diagonal entries, then the strictly-lower complex entries column by
 *                        column ((1,0) (2,0) .. (2N-1,0) (2,1) ..) as re,im — 16 reals (fundamental), 36 (adjoint);
 *                        block index = (spin mod 2)*N + colour
 *     "device layout" = the library's parity-split, x3-row-blocked structure of arrays;
 *     opaque to the caller except through hr_pack_* / hr_unpack_*.  A full-lattice device field is the
 *     even half followed by the odd half, each hr_*_bytes(geom, 0) long, so `field + half` is the odd half.
 *   - Lattice extents must be even and >= 2 (odd extents break the even-odd colouring under wrap-around).
 */
#ifndef HR_DSLASH_H
#define HR_DSLASH_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { HR_OK = 0, HR_EINVAL = 1, HR_EUNSUPPORTED = 2, HR_EALIGN = 3, HR_ECUDA = 4 };

/* fermion representation / gauge group.  HR_REP_FUND and HR_REP_ADJ are the two SU(2) representations of BASELINE.json;
 * HR_REP_SU3 is the first step towards HiRep's other gauge groups: 3 complex
 * colours and complex 3 x 3 links (canonical [V][4 mu][3][3][re,im]) kept on the device in full (link_storage = HR_LINKS_FULL, 18 reals)
 * or as their first two rows (HR_LINKS_COMPRESSED, 12 reals: the kernels and hr_unpack_gauge rebuild row 2 = conj(row 0 x row 1),
 * exact for unitary links of determinant 1).  It is
 * served by the generic hopping kernel: bare hops, full D, the even-odd operator with and without clover, the clover-improved full
 * operator, the clover block builders (regular and exponential; hr_clover_build takes the SU(3) gauge field itself as u_fund;
 * blocks are 6 x 6 like the adjoint ones), hr_clover_apply, the CG solvers and the sharded hop with every epilogue;
 * hr_represent_gauge (the SU(2) adjoint) returns HR_EUNSUPPORTED for it, hr_represent_gauge_antisym builds its two-index
 * antisymmetric representation. */
enum { HR_REP_FUND = 0, HR_REP_ADJ = 1, HR_REP_SU3 = 2 };
enum { HR_PREC_F64 = 0, HR_PREC_F32 = 1 };
/* fundamental links are stored as their first row (alpha, beta): U = [[alpha, beta], [-conj(beta), conj(alpha)]]
 * is exact for SU(2).  HR_LINKS_FULL (all four entries) is declared for the byte model only and is
 * rejected with HR_EUNSUPPORTED by the kernels. */
enum { HR_LINKS_FULL = 0, HR_LINKS_COMPRESSED = 1,
       /* adjoint fermions only: the operators are handed the FUNDAMENTAL (compressed) gauge field and rebuild the
        * real 3x3 link R^{ab} = 1/2 tr(sigma_a U sigma_b U^dag) in registers — 32 B instead of 72 B per fp64 link,
        * and no adjoint gauge field in memory ("higher representations") */
       HR_LINKS_ONTHEFLY = 2 };
/* which hopping kernel runs: AUTO picks the x0-marching tiled kernel when the lattice allows it and is
 * large enough to need it, else the generic one-thread-per-site kernel.  The other two values force a
 * kernel (HR_KERNEL_TILED fails with HR_EUNSUPPORTED if the lattice does not fit its tiles). */
enum { HR_KERNEL_AUTO = 0, HR_KERNEL_GENERIC = 1, HR_KERNEL_TILED = 2 };

typedef struct hr_geom {
    int L[4];         /* extents, L[0] = T (slowest) ... L[3] (fastest); all even, >= 2 */
    int rep;          /* HR_REP_*: representation of the FERMION (and of the links the operators read) */
    int prec;         /* HR_PREC_* : arithmetic and storage type of every field */
    int link_storage; /* HR_LINKS_*: FULL/COMPRESSED describe fundamental links; ONTHEFLY is for rep == HR_REP_ADJ */
    int kernel;       /* HR_KERNEL_* */
} hr_geom;

/* parity arguments */
enum { HR_EVEN = 0, HR_ODD = 1, HR_BOTH = 2 };

/* ---- sizes (host-only, no CUDA call).  0 is returned for an invalid geometry. ---- */
size_t hr_spinor_bytes(const hr_geom* g, int parity);      /* device layout; parity HR_EVEN/HR_ODD: half field, HR_BOTH: full */
size_t hr_gauge_bytes(const hr_geom* g, int rep);           /* device layout, all 4V links of representation `rep` */
size_t hr_clover_bytes(const hr_geom* g);                   /* device layout, one set of blocks (forward OR inverse), all V sites */
size_t hr_canonical_spinor_bytes(const hr_geom* g);         /* canonical, V sites */
size_t hr_canonical_gauge_bytes(const hr_geom* g, int rep); /* canonical, 4V links */
size_t hr_canonical_clover_bytes(const hr_geom* g);         /* canonical, V sites x 2 x (2N)^2 reals (N of g->rep) */

/* ---- canonical <-> device layout (both pointers on the device; pure permutations, no arithmetic) ---- */
int hr_pack_spinor(const hr_geom* g, const void* canon, void* dev, void* stream);
int hr_unpack_spinor(const hr_geom* g, const void* dev, void* canon, void* stream);
int hr_pack_gauge(const hr_geom* g, int rep, const void* canon, void* dev, void* stream);
int hr_unpack_gauge(const hr_geom* g, int rep, const void* dev, void* canon, void* stream);
int hr_pack_clover(const hr_geom* g, const void* canon, void* dev, void* stream);
int hr_unpack_clover(const hr_geom* g, const void* dev, void* canon, void* stream);

/* R1 (BASELINE.json north_star "Representation kernel"; "higher representations"):
 *   R^{ab}(x,mu) = 1/2 tr(sigma_a U_mu(x) sigma_b U_mu(x)^dag), a,b = 1..3, real 3x3, for all 4V links.
 * u_fund: fundamental gauge field, u_adj: adjoint gauge field, both device layout, sized by
 * hr_gauge_bytes(g, HR_REP_FUND / HR_REP_ADJ).  g->rep is ignored. */
int hr_represent_gauge(const hr_geom* g, const void* u_fund, void* u_adj, void* stream);

/* R1 for complex 3 x 3 links: the two-index antisymmetric representation (SURVEY.md §8(f) item 4 "symmetric/antisymmetric reps";
 * PAPER.md:21 "higher representations"; DESIGN.md §3 reading B9):
 *   R_ab(x,mu) = tr( e^a^dag U_mu(x) e^b U_mu(x)^T ),  e^a = (E_ij - E_ji)/sqrt(2) for the pairs a = (i<j) = (0,1), (0,2), (1,2),
 * i.e. the 2 x 2 minors of U (rows = pair a, columns = pair b), for all 4V links.  For three colours the representation is
 * three-dimensional and R is again special unitary, so u_rep has the layout and size of u_fund (hr_gauge_bytes(g, HR_REP_SU3),
 * all three rows with HR_LINKS_FULL, the first two with HR_LINKS_COMPRESSED) and every HR_REP_SU3 operator takes it as its gauge
 * field.  g->rep must be HR_REP_SU3 (else HR_EUNSUPPORTED); both pointers on the device, 16-byte aligned, not overlapping
 * (HR_EINVAL); the caller owns both; asynchronous on `stream`. */
int hr_represent_gauge_antisym(const hr_geom* g, const void* u_fund, void* u_rep, void* stream);

/* H3 (north_star "full form"): out = D psi on all V sites, one launch.
 * u: gauge field in representation g->rep (the fundamental field if g->link_storage == HR_LINKS_ONTHEFLY);
 * psi, out: full-lattice spinors (out must not alias psi). */
int hr_dirac_apply(const hr_geom* g, double m0, const void* u, const void* psi, void* out, void* stream);

/* H3c (north_star "optional clover-improved form"; "Clover improvement ... requires the application of
 * another diagonal term"): the clover-improved operator on all V sites in one launch,
 *     out = D_sw psi = A psi - 1/2 H psi,      A(x) = (4+m0) + C(x)  the forward blocks of hr_clover_build[_exp]
 * (m0 lives inside the blocks).  Both representations; out must not alias psi. */
int hr_dirac_clover_apply(const hr_geom* g, const void* u, const void* clover_fwd, const void* psi, void* out, void* stream);

/* H1/H2/E1/E2 (north_star "even-odd preconditioned form D_ee - D_eo D_oo^-1 D_oe as used in the HMC";
 * PAPER.md:39 "even-odd preconditioned version of the Dirac operator used mainly in the HMC").
 *   op = HR_EO_HOP_OE : out_o = H_oe in_e   (bare hopping sum, no -1/2), in: even half field, out: odd half field
 *   op = HR_EO_HOP_EO : out_e = H_eo in_o
 *   op = HR_EO_DHAT   : out_e = Dhat in_e, in and out even half fields, tmp an odd half field;
 *        without clover (clover_fwd == clover_inv == NULL):
 *              Dhat = (4+m0) - H_eo H_oe / (4 (4+m0))
 *        with clover (both non-NULL, built by hr_clover_build[_exp] with the same m0, for g->rep):
 *              Dhat = A_ee - 1/4 H_eo A_oo^-1 H_oe            (m0 is then ignored: it lives inside A)
 *        Two dependent launches on `stream` (the paper's "impossible to parallelise" pair of halves).
 * out must not alias in; tmp must alias neither. */
enum { HR_EO_HOP_OE = 0, HR_EO_HOP_EO = 1, HR_EO_DHAT = 2 };
int hr_dirac_eo_apply(const hr_geom* g, int op, double m0, const void* u, const void* clover_fwd,
                      const void* clover_inv, const void* in, void* out, void* tmp, void* stream);

/* E1/E2 without any device allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it):   out_e = Dhat in_e   exactly as hr_dirac_eo_apply(op = HR_EO_DHAT) computes
 * it (same kernels, same bits), with the odd half field between the two hops kept in a file-scope device array of the
 * library instead of a caller-owned `tmp`.  u, clover_fwd, clover_inv (both NULL or both given), in, out: device,
 * caller-owned, as for hr_dirac_eo_apply.
 *   - Limit: hr_spinor_bytes(g, HR_ODD) <= HR_STATIC_SCRATCH_BYTES (8 MiB: 16^3 x 32 SU(2)-fundamental sites in fp64,
 *     twice that in fp32); a larger lattice returns HR_EINVAL with the two sizes in hr_last_error() and launches nothing.
 *   - The call makes no cudaMalloc / cudaFree and calls no allocating library routine.  Every GPU that loads the library
 *     holds the 8 MiB until the process exits.  The first call on a device looks the array's device address up
 *     (cudaGetSymbolAddress, once per device, the device of `stream` current): make that call outside stream capture.
 *   - All calls on one device share the array, which keeps the last call's contents.  Nothing in it has to start at
 *     zero (the first hop writes every entry the second one reads), but two calls that overlap on the GPU — different
 *     streams, or graphs replayed concurrently — race on it: serialise them (one stream, or an event between them). */
#define HR_STATIC_SCRATCH_BYTES (8u << 20)
int hr_dhat_apply_static(const hr_geom* g, double m0, const void* u, const void* clover_fwd, const void* clover_inv,
                         const void* in, void* out, void* stream);

/* C1 ("precomputing certain fields ... recomputed whenever the gauge field is updated"):
 * from the FUNDAMENTAL gauge field build, for every site, the two hermitian chirality blocks (4x4 for fundamental
 * fermions, 6x6 for adjoint ones: g->rep, the leaves mapped to the adjoint representation) of
 *   A(x) = (4+m0) + csw (i/4) sum_{mu,nu} sigma_mu,nu F^_mu,nu(x)      (F^ from the four-leaf clover)
 * into clover_fwd and their inverses into clover_inv (either may be NULL to skip it).  Setup step. */
int hr_clover_build(const hr_geom* g, double m0, double csw, const void* u_fund, void* clover_fwd,
                    void* clover_inv, void* stream);

/* C1x ("exponential of the clover term"; ref [6] at PAPER.md:123): the same
 * block fields for the EXPONENTIAL clover improvement,
 *   A_exp(x) = (4+m0) exp( C(x) / (4+m0) ),   A_exp(x)^-1 = exp( -C(x) / (4+m0) ) / (4+m0),
 * C(x) = csw (i/4) sum_{mu,nu} sigma_mu,nu F^_mu,nu(x) as above (the regular term (4+m0) + C is its first two
 * orders).  hr_clover_apply and hr_dirac_eo_apply take these blocks unchanged; forward and inverse blocks cost the
 * same to apply, as the paper notes.  Setup step; arithmetic in double for either field precision. */
int hr_clover_build_exp(const hr_geom* g, double m0, double csw, const void* u_fund, void* clover_fwd,
                        void* clover_inv, void* stream);

/* C2/C3 ("application of another diagonal term"): out(x) = B(x) in(x) on the sites of
 * `parity` (HR_EVEN, HR_ODD: in/out are half fields; HR_BOTH: full fields).  `blocks` is the full-lattice
 * block field (forward blocks: C2; inverse blocks: C3 — same kernel).  Both representations. */
int hr_clover_apply(const hr_geom* g, int parity, const void* blocks, const void* in, void* out, void* stream);
/* Number of non-finite reals in a block field (forward or inverse), written as one unsigned 64-bit integer to
 * count_dev (device memory, 8-byte aligned, caller-owned; read it after synchronising the stream).  The inverse blocks
 * are made by Gauss-Jordan elimination with partial pivoting in double precision: accurate whenever A(x) is
 * invertible (it is positive definite for |csw F| < 4+m0, the regime of BASELINE.json configs[4]); an exactly
 * singular A(x) gives inf / nan entries, which this call counts — 0 means every block is usable. */
int hr_clover_count_nonfinite(const hr_geom* g, const void* blocks, void* count_dev, void* stream);

/* M1 ("measured in terms of memory bandwidth"): the work model, per OUTPUT site of `op`,
 * for the storage described by g.  bytes_compulsory: every distinct datum crosses DRAM once per kernel;
 * bytes_requested: no reuse at all (every neighbour spinor counted), the paper-style figure. Host-only. */
enum {
    HR_OP_HOP = 0,        /* bare parity hop H1                     */
    HR_OP_DIRAC = 1,      /* full D, one launch (H3), per site of V */
    HR_OP_DHAT = 2,       /* E1, per even site                      */
    HR_OP_CLOVER = 3,     /* C2/C3                                  */
    HR_OP_DHAT_CLOVER = 4,/* E2, per even site                      */
    HR_OP_REPRESENT = 5   /* R1, per site (4 links)                 */
};
int hr_dirac_flops_bytes(const hr_geom* g, int op, double* flops_per_site, double* bytes_compulsory,
                         double* bytes_requested);

/* S1 ("a range of inverters", PAPER.md:39 the even-odd operator is the one
 * "used mainly in the HMC"): conjugate gradient on the normal equations of the even-odd operator,
 *       Dhat^dag Dhat x = b      on the even sites,      Dhat^dag = gamma5 Dhat gamma5,
 * Dhat as in hr_dirac_eo_apply(op = HR_EO_DHAT) (with clover if both block fields are given), started from x = 0,
 * textbook Hestenes-Stiefel recurrences in the field precision with double-precision, fixed-order reductions.
 * Stops when |r| <= tol |b| or after max_iter iterations; the residual is read back every check_every iterations
 * (so up to check_every - 1 extra iterations are made) — the one call of this library that synchronises `stream`.
 *   b, x: even half fields (device); workspace: device, hr_cg_workspace_bytes(g) bytes; iters, relres: HOST
 *   outputs (may be NULL): iterations made and the recurrence residual |r|/|b|.
 * Returns HR_OK also when max_iter was reached without convergence (check *relres). */
size_t hr_cg_workspace_bytes(const hr_geom* g);
int hr_cg_solve(const hr_geom* g, double m0, const void* u, const void* clover_fwd, const void* clover_inv,
                const void* b, void* x, void* workspace, double tol, int max_iter, int check_every,
                int* iters, double* relres, void* stream);

/* S2 ("mixed fp32/fp64 defect correction"): the same system solved to double-precision
 * accuracy with the iterations done in single precision.  Outer loop (fp64): r = b - Dhat^dag Dhat x evaluated with
 * the fp64 operator; stop when |r| <= tol |b| (this is the TRUE residual) or after max_outer corrections; otherwise
 * solve Dhat^dag Dhat e = r with hr_cg_solve's iteration on the fp32 fields to the relative accuracy inner_tol
 * (at most max_inner iterations), x += e.  g describes the fp64 fields (prec = HR_PREC_F64);
 * u_f64 / u_f32: the SAME gauge field packed in both precisions; b, x: fp64 even half fields;
 * workspace: hr_cg_mixed_workspace_bytes(g).  HOST outputs (may be NULL): corrections made, total fp32 iterations,
 * final true |r|/|b|.  Synchronises `stream` once per outer iteration (and as hr_cg_solve inside). */
size_t hr_cg_mixed_workspace_bytes(const hr_geom* g);
int hr_cg_solve_mixed(const hr_geom* g, double m0, const void* u_f64, const void* u_f32, const void* b, void* x,
                      void* workspace, double tol, double inner_tol, int max_outer, int max_inner, int check_every,
                      int* outer_iters, int* inner_iters, double* relres, void* stream);
/* the same with the clover-improved operator: the block fields of hr_clover_build[_exp] in both precisions */
int hr_cg_solve_mixed_clover(const hr_geom* g, double m0, const void* u_f64, const void* u_f32,
                             const void* clover_fwd_f64, const void* clover_inv_f64, const void* clover_fwd_f32,
                             const void* clover_inv_f32, const void* b, void* x, void* workspace, double tol,
                             double inner_tol, int max_outer, int max_inner, int check_every, int* outer_iters,
                             int* inner_iters, double* relres, void* stream);

/* ---- host-buffer entry points (the end-to-end path a user without device buffers calls) ----
 * All data pointers are HOST pointers to canonical arrays (pinned memory makes the copies asynchronous);
 * `workspace` is a DEVICE buffer of at least hr_host_workspace_bytes(g) bytes.  The call uploads gauge
 * and spinor, packs, applies, unpacks, downloads, and synchronises `stream` before returning.
 *   hr_dirac_apply_host    : out[V] = D psi[V]
 *   hr_dirac_eo_apply_host : op as in hr_dirac_eo_apply without clover; full-lattice canonical arrays: only the
 *                            entries of the input parity are read; ALL of out is written — the entries of the
 *                            output parity with the result, those of the other parity with zeros. */
size_t hr_host_workspace_bytes(const hr_geom* g);
int hr_dirac_apply_host(const hr_geom* g, double m0, const void* u_canon_host, const void* psi_canon_host,
                        void* out_canon_host, void* workspace, void* stream);
int hr_dirac_eo_apply_host(const hr_geom* g, int op, double m0, const void* u_canon_host,
                           const void* in_canon_host, void* out_canon_host, void* workspace, void* stream);

/* ---- the sharded hop: one rank of a 4-D domain decomposition (§2.1 "inner computations
 * ... boundary calculation ... send buffer", Fig. 4 "all four dimensions parallelized").
 * g describes the rank's LOCAL lattice (ordinary device layout); hr_decomp says which directions are cut between ranks.
 * Across a cut the hopping sum needs the neighbour rank's boundary spinors; they travel as FACES of spin-projected
 * half spinors (2N complex numbers per face site instead of 4N; the backward face is already multiplied by the
 * sender's link, so links never move):
 *   face index 2*mu   "down": the sender's sites with x_mu = 0,        (1 - gamma_mu) psi projected; goes to the rank at -mu
 *   face index 2*mu+1 "up"  : the sender's sites with x_mu = L_mu - 1, U_mu^dag (1 + gamma_mu) psi;   goes to the rank at +mu
 * A face holds the sites of one parity (the hop's input parity) indexed by the other three coordinates, in 16-byte
 * chunks [chunk][face site]; hr_halo_face_bytes(g, mu) bytes, opaque to the caller, 16-byte aligned.
 *   hr_halo_pack : writes the 2 faces of every cut direction from the half field `in_half` of parity in_parity.
 *                  face_out[8] (host array of device pointers, entries of uncut directions ignored) may point into the
 *                  neighbour's receive buffer when that memory is peer-mapped (NVLink): then packing IS the transfer.
 *   hr_hop_local : out_half (parity out_parity) = epilogue( H in_half ) on the local lattice: an interior kernel that
 *                  leaves out the terms crossing a cut, then one boundary kernel per received face that adds them.
 *                  face_in[2*mu] = the down face of the rank at +mu, face_in[2*mu+1] = the up face of the rank at -mu.
 *                  epi / a / c / clover / phi_half as the epilogues of the single-GPU hop:
 *                    HR_EPI_NONE        out = H in                      HR_EPI_AXPY        out = a phi + c H in
 *                    HR_EPI_CLOVER_INV  out = B (H in)                  HR_EPI_CLOVER_AXPY out = B phi + c H in
 *                  (B = the blocks of `clover`, a full-lattice block field).  With no cut direction this is the
 *                  single-GPU hop.  The transfer between pack and hop is the caller's (NCCL send/recv, peer copies):
 *                  Dhat = hop, exchange, hop — see paper_2411_18511_b200/halo.py for the composition. */
typedef struct hr_decomp {
    int split[4];   /* split[mu] != 0: direction mu is cut between ranks; 0: periodic inside the local lattice */
} hr_decomp;
enum { HR_EPI_NONE = 0, HR_EPI_AXPY = 1, HR_EPI_CLOVER_INV = 2, HR_EPI_CLOVER_AXPY = 3 };
size_t hr_halo_face_bytes(const hr_geom* g, int mu);
int hr_halo_pack(const hr_geom* g, const hr_decomp* d, int in_parity, const void* u, const void* in_half, void* const* face_out, void* stream);
int hr_hop_local(const hr_geom* g, const hr_decomp* d, int out_parity, int epi, double a, double c, const void* u, const void* clover,
                 const void* in_half, const void* phi_half, void* out_half, const void* const* face_in, void* stream);
/* The two halves of hr_hop_local, for overlapping the face transfer with the interior kernel ("the inner Dirac
 * kernel ... [while] the communications take place"): enqueue hr_halo_pack and the transfer on one stream, the interior on
 * another, make the second stream wait for the transfer, then enqueue the boundary part (paper_2411_18511_b200/halo.py:
 * hop_all(overlap=True)).  Same arguments as hr_hop_local; the boundary part needs neither in_half nor phi_half. */
int hr_hop_local_interior(const hr_geom* g, const hr_decomp* d, int out_parity, int epi, double a, double c, const void* u, const void* clover,
                          const void* in_half, const void* phi_half, void* out_half, void* stream);
int hr_hop_local_boundary(const hr_geom* g, const hr_decomp* d, int out_parity, int epi, double c, const void* u, const void* clover,
                          void* out_half, const void* const* face_in, void* stream);

/* ---- host path with the gauge field resident on the device ----
 * The gauge field changes once per molecular-dynamics step and the operator is applied many times in between
 * (PAPER.md:53-59): upload the links once, then stream right-hand sides through.
 *   hr_gauge_upload_host : canonical host links (rep = HR_REP_FUND: [lex][mu][2][2][re,im]; HR_REP_ADJ: [lex][mu][3][3])
 *                          -> device layout in u_dev (hr_gauge_bytes(g, rep)); workspace = hr_canonical_gauge_bytes(g, rep)
 *                          device bytes.  Synchronises `stream` before returning.
 *   hr_apply_host_batch  : out_i = Op in_i for i = 0 .. nrhs-1, canonical full-lattice arrays in host memory (pinned
 *                          memory for full PCIe speed; the two pointer arrays live in host memory).  op = HR_EO_HOP_OE,
 *                          HR_EO_HOP_EO, HR_EO_DHAT (as hr_dirac_eo_apply_host: entries of the other parity are not
 *                          read and come back as zeros; with clover_fwd and clover_inv the clover-improved operator E2)
 *                          or HR_HOST_DIRAC (full D; with clover_fwd the clover-improved D_sw; clover_inv must be NULL).
 *                          Three-stage pipeline over two library-owned copy streams (created per device on first use
 *                          and kept for the life of the process — the one place this library allocates anything) and
 *                          the caller's stream: upload of spinor i+1, pack + operator + unpack of spinor i and download
 *                          of result i-1 overlap, so both PCIe directions are busy.  workspace =
 *                          hr_host_batch_workspace_bytes(g) device bytes.  Returns after the last result has arrived.
 *   hr_apply_host_ops    : the same pipeline with one operator PER ITEM (ops[i], same codes): out_i = Op_i in_i.  A sequence of
 *                          different operators then pays the pipeline's fill and drain (one upload and one download that overlap
 *                          nothing) once, not once per operator.  With clover blocks the HR_EO_DHAT items use clover_fwd and
 *                          clover_inv, the HR_HOST_DIRAC items clover_fwd. */
enum { HR_HOST_DIRAC = 3 };
int hr_gauge_upload_host(const hr_geom* g, int rep, const void* u_canon_host, void* u_dev, void* workspace, void* stream);
size_t hr_host_batch_workspace_bytes(const hr_geom* g);
int hr_apply_host_ops(const hr_geom* g, const int* ops, double m0, const void* u_dev, const void* clover_fwd, const void* clover_inv,
                      int nitems, const void* const* in_canon_host, void* const* out_canon_host, void* workspace, void* stream);
int hr_apply_host_batch(const hr_geom* g, int op, double m0, const void* u_dev, const void* clover_fwd, const void* clover_inv,
                        int nrhs, const void* const* in_canon_host, void* const* out_canon_host, void* workspace, void* stream);

/* ---- diagnostics ---- */
size_t hr_last_error(char* buf, size_t len);   /* copies the last error text (NUL-terminated); returns its length */
/* number of kernels this library has launched since load (bench.py's gpu_launches) */
unsigned long long hr_launch_count(void);
/* name of the hopping kernel hr_dirac_eo_apply/hr_dirac_apply would run for g: "generic" or "tiled" */
const char* hr_kernel_name(const hr_geom* g);
/* The launch plan of the kernel behind op = HR_OP_HOP (a parity hop, also each hop of HR_OP_DHAT) or HR_OP_DIRAC
 * (hr_dirac_apply) on the calling thread's current device; host only, nothing is launched.  info[8] receives
 *   [0] kernel: 0 generic (the rest is then 0), 1 hop_tiled_kernel, 2 dirac_tiled_kernel
 *   [1],[2] tile shape T1 x T2 in x3-rows   [3] x0 segments per tile   [4] planes per segment (L0 / segments)
 *   [5] threads per CTA   [6] dynamic shared memory in bytes   [7] CTAs in the grid.
 * For tests (which segment lengths a lattice exercises) and for the profile notes; other ops return HR_EINVAL. */
int hr_kernel_plan(const hr_geom* g, int op, int* info);

#ifdef __cplusplus
}
#endif
#endif /* HR_DSLASH_H */
