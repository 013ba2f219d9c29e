/*
 * cola.h -- C ABI of the B200-native COLA hot path (libcola.so).
 *
 * What it is.  The paper (arxiv 2302.00850, PAPER.md; "P:n" = line n) describes a GPU "fermion
 * matrix inverter" (conjugate gradient, mixed precision: 32-bit inner, 64-bit outer),
 * one lattice site per thread, written in CUDA and called from Fortran through ISO-C-binding
 * C-callable routines.  This header is that boundary.  The operator is fixed by
 * BASELINE.json north_star (BJ:ns) and written out in SURVEY.md section 8(c) O1..O8 / DESIGN.md:
 *
 *     M = A - kappa*D                                  Wilson-clover, kappa normalisation, r = 1
 *     (D psi)(x) = sum_mu [ eta+ (1-gamma_mu) U_mu(x) psi(x+mu) + eta- (1+gamma_mu) U_mu(x-mu)^+ psi(x-mu) ]
 *     A(x) = 1 - kappa*csw*sum_{mu<nu} sigma_{mu nu} F_{mu nu}(x)     (two 6x6 Hermitian chiral blocks)
 *     S = A_ee - kappa^2 D_eo A_oo^{-1} D_oe           even-odd Schur complement on even sites
 *     K^+ = gamma_5 K gamma_5 for K = M, S
 *
 * General rules.
 *   - No torch types, no C++ types: plain pointers and sizes.  Every pointer argument says whether
 *     it is a HOST or a DEVICE pointer.  Device memory is owned by the caller (PyTorch tensors);
 *     the library allocates no device memory except a 4 KB control block: gauge field, clover
 *     field and solver vectors live in the caller-provided workspace (cola_set_workspace), which
 *     the context borrows until cola_destroy / the next cola_set_workspace.
 *   - Every function returns a cola_status and never throws or aborts across the ABI; a message
 *     for the last failure on a context is available from cola_last_error.
 *   - Operator applications are asynchronous on the context's stream.  cola_gauge_upload*,
 *     cola_cg_solve* and every *_host entry point synchronise that stream before returning.
 *   - Lattice: dims = (Lx, Ly, Lz, Lt), each even and >= 2.  V = Lx*Ly*Lz*Lt, Vh = V/2.
 *     Site index i(x) = x + Lx*(y + Ly*(z + Lz*t)); parity = (x+y+z+t) mod 2 (0 = even).
 *   - Canonical arrays (what the caller sees), complex = (re, im) pairs, C order:
 *         links   U[t][z][y][x][mu][a][b]   fp64     (U psi)_a = sum_b U_ab psi_b, mu = x,y,z,t
 *         spinor  psi[t][z][y][x][s][c]     fp64 or fp32 (complex128 / complex64)
 *         clover  A[t][z][y][x][12][12]     fp64, row = 3*s + c
 *   - Internal arrays (what the kernels see): parity-split structure of arrays of 16-byte chunks,
 *     site index fastest:   spinor[parity][chunk][Vh]  with chunk = 2 (fp64) or 4 (fp32) reals,
 *     24 reals per site in canonical (s, c, re/im) order.  A "half-lattice" internal buffer is one
 *     parity of that (cola_spinor_bytes(.., full=0) bytes); a full internal buffer is the even
 *     half followed by the odd half.
 */
#ifndef COLA_H
#define COLA_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cola_ctx cola_ctx;   /* opaque; created by cola_create, owned by the library */

typedef enum {
    COLA_OK = 0,
    COLA_EINVAL = 1,     /* bad argument (odd extent, NULL pointer, non-unitary links with compress12, ...) */
    COLA_ECUDA = 2,      /* a CUDA call or kernel failed; cola_last_error has the CUDA message */
    COLA_ENOTREADY = 3,  /* operator/solver called before cola_set_workspace + cola_gauge_upload */
    COLA_ENOCONV = 4,    /* cola_cg_solve hit max_iter; info is filled, x holds the last iterate */
    COLA_ENOMEM = 5      /* workspace too small */
} cola_status;

/* COLA_F32_H16 ("additional computation in order to reduce traffic", P:45 mixed precision):
 * fp32 spinors and fp32 arithmetic, but links read from 16-bit fixed point (12 reals, third row rebuilt) and the
 * clover fields from fp16, which cuts the bytes per Schur application from 1824 to 1152 per site.  It is an
 * approximate ("sloppy") operator, |K16 x - K x| / |K x| ~ 1e-4, meant for the inner iteration of the mixed-precision
 * solver (cola_solve_params.mixed = 2), whose reliable updates use the exact fp64 operator.  Spinor buffers and
 * cola_spinor_* calls take COLA_F32 for it. */
/* COLA_F32_R8 (the rest of SURVEY 8(f) NEXT-2): fp32 spinors and arithmetic, links read as 8 fp32 reals (a
 * parametrisation of SU(3): two entries of row 1, one of column 1 and two phases; the other entries follow from unitarity
 * and det U = 1 in registers): 1472 bytes per Schur application and site instead of 1728.  Like COLA_F32 (when
 * trace_sub = 1) it reads A in its 48-real field-strength form: per chiral block the three traceless Hermitian 3x3 matrices
 * of  1 + [[G3, G1 - i G2], [G1 + i G2, -G3]], expanded to the packed 6x6 block in the kernel (192 instead of 288 bytes).  The same linear map as COLA_F32 up to rounding (sin/cos, 1/x and sqrt are the
 * hardware approximations: a link entry is good to ~4e-7 absolute); the parity tests hold
 * it to the fp32 tolerance 2e-6.  Needs COLA_FEAT_R8 and links unitary to 1e-10 with every |U00| >= 0.1
 * (cola_gauge_info_r8), else COLA_EINVAL.  Measured on B200 the 8-real links do not pay (the kernels become bound on the SM
 * side: +7-10 % time for -13 % bytes); the format is kept as an option.
 * cola_solve_params.mixed = 3 runs the inner iteration on it.  Spinor buffers and cola_spinor_* calls take COLA_F32. */
typedef enum { COLA_F64 = 0, COLA_F32 = 1, COLA_F32_H16 = 2, COLA_F32_R8 = 3 } cola_prec;
typedef enum { COLA_EVEN = 0, COLA_ODD = 1 } cola_parity;

typedef struct {
    int dims[4];        /* Lx, Ly, Lz, Lt: each even, >= 2 */
    double kappa;       /* hopping parameter */
    double csw;         /* clover coefficient */
    int bc[4];          /* +1 periodic / -1 antiperiodic per direction; the configs use {+1,+1,+1,-1} */
    int compress12;     /* 1: fp32 links stored as 12 reals, third row rebuilt in registers (BJ:ns);
                           0: fp32 links stored as 18 reals.  fp64 links are always 18 reals. */
    int trace_sub;      /* 1 (default reading): remove the trace of F_{mu nu} */
    int device;         /* CUDA device ordinal */
    void *stream;       /* cudaStream_t to launch on (e.g. torch.cuda.current_stream().cuda_stream); NULL = default */
} cola_params;

/* Create a context for one lattice.  HOST pointers.  COLA_EINVAL for odd / too small extents or
 * bc not in {+1,-1}; COLA_ECUDA if the device cannot be selected. */
cola_status cola_create(cola_ctx **out, const cola_params *p);
cola_status cola_destroy(cola_ctx *c);
/* Message of the last failure on c (valid until the next call on c); "" if none.  c may be NULL
 * (returns the message of the last failed context-free call -- cola_create, cola_spinor_norm2_static -- in this thread). */
const char *cola_last_error(const cola_ctx *c);
/* Tuning: bytes of L2 the kernels' sweep order may count on for the reuse of neighbour spinors (default 40 MB; 0
 * restores it).  A neighbour spinor is used from three consecutive time slices; when three slices of reused spinors
 * (all right-hand sides of a launch) exceed this budget the thread blocks sweep the lattice in bands of z-planes
 * instead of slice by slice, which keeps the reuse inside L2.  Results do not depend on it. */
cola_status cola_set_l2_budget(cola_ctx *c, size_t bytes);
/* Optional parts of the workspace (the fields are ~8.0 KB per even site with everything on: 134 GB at 64^3x128).
 * Call before cola_workspace_bytes / cola_set_workspace (it un-lends the workspace and invalidates the gauge field).
 * Default: COLA_FEAT_ALL.
 *   COLA_FEAT_FULL_M  fp32 (and fp16) copies of A on the ODD parity and the larger solver scratch: needed by
 *                     cola_fermion_matrix_apply* in COLA_F32 / COLA_F32_H16 and by solves with even_odd = 0.  The fp64
 *                     operator on the full lattice is always available (the true residual |b - M x| needs it).
 *   COLA_FEAT_H16     16-bit links + fp16 clover: COLA_F32_H16 operators and mixed = 2.
 *   COLA_FEAT_R8      8-real fp32 links: COLA_F32_R8 operators and mixed = 3.
 *   COLA_FEAT_A72     the fp32 copy of A as packed 6x6 blocks (72 reals).  The fp32 kernels read A in its 48-real
 *                     field-strength form (see COLA_F32_R8 above; -10 % bytes on M, measured -9 % time); the 72-real copy is
 *                     only read after cola_set_compact cleared bit 1 (A/B measurements) and is always carved when
 *                     trace_sub = 0, where the 48-real form does not exist.
 * A call that needs a missing feature returns COLA_EINVAL. */
typedef enum { COLA_FEAT_FULL_M = 1, COLA_FEAT_H16 = 2, COLA_FEAT_R8 = 4, COLA_FEAT_A72 = 8, COLA_FEAT_ALL = 15 } cola_feature;
cola_status cola_set_features(cola_ctx *c, unsigned features);
/* Change the stream subsequent calls launch on. */
cola_status cola_set_stream(cola_ctx *c, void *stream);

/* Bytes of one internal spinor buffer: full != 0 -> V sites, else Vh sites. */
size_t cola_spinor_bytes(const cola_ctx *c, cola_prec prec, int full);
/* Bytes of workspace the context needs (gauge fp64 + fp32, clover A both parities and A^-1 on the
 * odd parity in fp64 + fp32, solver vectors, staging). */
size_t cola_workspace_bytes(const cola_ctx *c);
/* Lend `bytes` of DEVICE memory (256-byte aligned) to the context.  COLA_ENOMEM if too small.
 * Invalidates a previously uploaded gauge field. */
cola_status cola_set_workspace(cola_ctx *c, void *dev_ptr, size_t bytes);

/* H0-H2: upload canonical fp64 links, reorder to the internal parity-split SoA
 * (fp64 18 reals; fp32 18 or 12 reals), build the clover field A from the four-leaf field
 * strength, invert its 6x6 blocks on the odd parity, make fp32 copies.  Links stay pure SU(3)
 * (no boundary sign folded in).  host_links: HOST pointer, 4*V*18 doubles.
 * With compress12, links with max|U U^+ - 1| > 1e-10 are rejected with COLA_EINVAL.  Without compress12 such links
 * are accepted for the fp64 and fp32 x18 operators, but their 16-bit copy (always 12 reals, third row rebuilt) would be
 * wrong: COLA_F32_H16 operators and mixed = 2 solves then return COLA_EINVAL.
 * COLA_EINVAL also if a 6x6 block of A on the odd parity is not positive definite (a Gauss-Jordan pivot <= 0;
 * SURVEY O6 expects eigenvalues in about [0.74, 1.26] for the configs): the Schur complement needs A_oo^-1. */
cola_status cola_gauge_upload(cola_ctx *c, const double *host_links);
/* Same, from a DEVICE pointer (e.g. links generated on the GPU for the 64^3x128 case). */
cola_status cola_gauge_upload_dev(cola_ctx *c, const double *dev_links);
/* Diagnostics of the last upload: max |U U^+ - 1| over all links. */
cola_status cola_gauge_info(const cola_ctx *c, double *max_unitarity_dev);
/* Diagnostics of the last upload for COLA_F32_R8: the smallest |U00| over all links.  The 8-real format rebuilds
 * |U00| = sqrt(1 - |U01|^2 - |U02|^2), whose absolute error grows like eps/(2 |U00|); it is offered only when every
 * |U00| >= 0.1 (true of the smooth ensembles of the configs, not of Haar-random links). */
cola_status cola_gauge_info_r8(const cola_ctx *c, double *min_abs_u00);
/* Diagnostics of the last upload (SURVEY O6 "report the smallest pivot it meets"): the smallest pivot of the unpivoted
 * Gauss-Jordan inversions of the 6x6 blocks of A_oo.  Valid (and <= 0) also after an upload that failed for it. */
cola_status cola_clover_info(const cola_ctx *c, double *min_pivot);

/* Tests of H1/H2: expand the packed fp64 clover field to canonical 12x12 blocks.
 * which = 0: A on all sites.  which = 1: A^-1 on odd sites, zero blocks on even sites.
 * canon_dev: DEVICE pointer, V*144 complex128. */
cola_status cola_clover_unpack(cola_ctx *c, int which, void *canon_dev);

/* Canonical DEVICE spinor (complex128 for COLA_F64, complex64 for COLA_F32) <-> full internal
 * DEVICE buffer of the same precision. */
cola_status cola_spinor_pack(cola_ctx *c, cola_prec prec, const void *canon_dev, void *internal_dev);
cola_status cola_spinor_unpack(cola_ctx *c, cola_prec prec, const void *internal_dev, void *canon_dev);
/* Internal fp64 <-> internal fp32 (round to nearest even), n_half = 1 (half lattice) or 2 (full).
 * cola_spinor_pack / unpack / convert take COLA_F64 or COLA_F32 only (COLA_EINVAL otherwise). */
cola_status cola_spinor_convert(cola_ctx *c, cola_prec dst_prec, const void *src_dev, void *dst_dev, int n_half);

/* ---- |v|^2 of an internal spinor buffer (the reduction of the fused BLAS-1 layer on its own).
 * The sum is accumulated in fp64 also for fp32 vectors and is bitwise reproducible: warp shuffle, block, then the last
 * thread block to finish adds the per-block partials in index order.  Asynchronous on the context's stream.
 *   v_dev    DEVICE, internal buffer of precision prec (COLA_F64 or COLA_F32); n_half = 1: one half lattice, 2: full
 *   out_dev  DEVICE, one double
 * The per-block partials and the tickets of the reduction live in the workspace lent to the context: COLA_ENOTREADY
 * without one.  No gauge field is needed. */
cola_status cola_spinor_norm2(cola_ctx *c, cola_prec prec, const void *v_dev, int n_half, double *out_dev);

/* The same |v|^2 for callers that cannot allocate device memory at all -- the only entry point of this library that needs
 * neither a context (cola_create allocates a control block and pinned host memory) nor a lent workspace (someone has to
 * allocate that too).  Who that is: code that is handed device pointers by a host application and nothing else, e.g.
 * a callback running after the application's memory pool has claimed the whole GPU, so that a raw cudaMalloc would
 * report out-of-memory; or a monitoring hook in a time-critical loop, where cudaMalloc / cudaFree are unwelcome
 * because they synchronise the whole device.  Such a caller can still measure a source or a residual with this call.
 *
 * It runs the kernel of cola_spinor_norm2 with the reduction's scratch (per-block partials, tickets) in a fixed
 * COLA_STATIC_SCRATCH_BYTES (16 KB) array that is part of libcola.so's device image: every GPU that loads the library
 * carries it until the process exits.  The call itself performs no cudaMalloc, cudaFree or other allocating call; it
 * issues one 36-byte cudaMemsetAsync (the tickets must start from zero, whatever an earlier call left behind) and one
 * kernel on `stream`.  The result equals cola_spinor_norm2's bit for bit (same grid, same summation order).
 *   device   CUDA device ordinal (0..63) the pointers belong to; made current for the call, the caller's device is restored
 *   stream   cudaStream_t of that device to launch on, NULL = default stream.  Asynchronous: out_dev is valid once
 *            the stream has reached this point
 *   prec     COLA_F64 or COLA_F32
 *   v_dev    DEVICE, n_sites sites of an internal buffer, i.e. 24 * n_sites reals, 16-byte aligned, owned by the caller
 *   n_sites  1 .. COLA_STATIC_MAX_SITES (2^25 = the full 64^3x128 lattice of the largest configuration; the call is
 *            tested up to that size and refuses more with COLA_EINVAL -- the scratch itself cannot overflow, the
 *            kernel's grid is capped at 1184 blocks)
 *   out_dev  DEVICE, one double, owned by the caller
 * First use: the first call on each device looks up that device's address of the array (cudaGetSymbolAddress) and
 * remembers it.  Make that first call during set-up, outside any stream capture.
 * Sharing: all calls in the process use the same array, and it keeps what the last call wrote.  Two calls whose
 * kernels can overlap on one GPU (different streams, different host threads) race on it and return garbage:
 * order them on one stream or with events.  Calls on different GPUs do not interact.
 * Errors: COLA_EINVAL (NULL pointer, n_sites = 0 or above the maximum, bad prec or device), COLA_ECUDA; the message is
 * available from cola_last_error(NULL) in the calling thread. */
#define COLA_STATIC_SCRATCH_BYTES 16384
#define COLA_STATIC_MAX_SITES 33554432
cola_status cola_spinor_norm2_static(int device, void *stream, cola_prec prec, const void *v_dev, size_t n_sites, double *out_dev);

/* H3-H5, parity dslash: out_p = D_{p,1-p} in_{1-p}.  in, out: internal half-lattice DEVICE buffers
 * (in holds parity 1-p, out receives parity p); they must not overlap. */
cola_status cola_dslash_apply(cola_ctx *c, cola_prec prec, cola_parity out_parity, const void *in_dev, void *out_dev);
/* H7: out = M in (dagger != 0: M^+ in).  Full internal DEVICE buffers, no overlap. */
cola_status cola_fermion_matrix_apply(cola_ctx *c, cola_prec prec, int dagger, const void *in_full_dev, void *out_full_dev);
/* H8: out_e = S in_e (dagger != 0: S^+).  Half-lattice (even) internal DEVICE buffers, no overlap.
 * Uses the context's odd half-lattice temporary. */
cola_status cola_schur_apply(cola_ctx *c, cola_prec prec, int dagger, const void *in_even_dev, void *out_even_dev);

typedef struct {
    double tol;        /* stop when |r| <= tol*|b| (1e-10 in the configs); r is the residual of the system
                          being iterated (M x = b, or S x_e = bhat_e whose residual equals the full one) */
    int max_iter;      /* CGLS passes (one K and one K^+ each) */
    int even_odd;      /* 0: CGNR on M (BJ:c0); 1: CGNR on the Schur complement + reconstruction */
    int mixed;         /* 0: all fp64; 1: fp32 inner iteration with fp64 reliable updates;
                          2: as 1, with the inner operator reading 16-bit links and clover (COLA_F32_H16);
                          3: as 1, with the inner operator reading 8-real links and the 48-real A (COLA_F32_R8) */
    double delta;      /* reliable-update threshold (mixed only); <= 0 selects the default 0.1 */
    int method;        /* COLA_CGNR (0, the north_star solver) or COLA_BICGSTAB: BiCGStab in van der
                          Vorst's order on the Schur system (needs even_odd = 1), x0 = 0, shadow residual = r0; one pass =
                          two applications of S (CGNR: S and S^+), `iters` counts passes.  COLA_EINVAL on breakdown
                          (<rhat, v> or rho vanishing).  t = S s = 0 is not one: the half step x + alpha p is then the
                          exact solution and the pass ends with omega = 0.  Mixed precision and reliable updates as for CGNR. */
} cola_solve_params;
typedef enum { COLA_CGNR = 0, COLA_BICGSTAB = 1 } cola_method;

typedef struct {
    int iters;                 /* CGLS passes done */
    int reliable_updates;      /* fp64 residual recomputations (mixed only) */
    double iterated_residual;  /* |r|/|b| of the recurrence (fp64 after the last reliable update) */
    double true_residual;      /* |b - M x|/|b| recomputed in fp64 on the full lattice */
    double seconds;            /* device time of the whole solve incl. source preparation and
                                  reconstruction, measured with CUDA events on the context's stream */
    double op_flops;           /* counted operator flops (1320/site dslash, 504/site clover, 48 xpay) */
} cola_solve_info;

/* H9-H12: solve M x = b.  b_canon_dev / x_canon_dev: canonical complex128 DEVICE arrays, V sites.
 * Returns COLA_OK, or COLA_ENOCONV with info filled and x = last iterate; COLA_EINVAL if the source (or, through the
 * residual, the gauge field) contains NaN or Inf. */
cola_status cola_cg_solve(cola_ctx *c, const cola_solve_params *sp, const void *b_canon_dev, void *x_canon_dev, cola_solve_info *info);

/* Same solve, also recording the residual history of the recurrence: resid_hist_host[k] = |r_{k+1}| / |b| after CGLS
 * pass k (k < min(info->iters, hist_len)); HOST array of hist_len doubles.  In the mixed modes this is the fp32
 * recurrence's residual (the value the reliable-update test sees), before a reliable update replaces it.
 * update_iters_host (HOST, may be NULL): receives the 1-based pass numbers after which the reliable updates fired
 * (the first min(info->reliable_updates, update_len) of them) -- SURVEY O8's schedule, compared in the tests with the
 * rule applied to the oracle's fp64 history. */
cola_status cola_cg_solve_history(cola_ctx *c, const cola_solve_params *sp, const void *b_canon_dev, void *x_canon_dev, cola_solve_info *info,
                                  double *resid_hist_host, int hist_len, int *update_iters_host, int update_len);

/* ---- Low modes of H = S^+ S on the even sites ("solvers for linear systems and eigenmodes",
 * ref [1] P:65) by thick-restart Lanczos on a Chebyshev polynomial of H, fp64, on the Schur kernels above.
 *   n_ev          eigenpairs wanted (the n_ev smallest eigenvalues of H), 1..32
 *   n_kr          dimension of the Krylov space kept between restarts, n_ev + 2 .. 64 (default when 0: 2 n_ev + 8)
 *   tol           stop when the residual estimate of every wanted Ritz pair of the filtered operator is <= tol times
 *                 its largest Ritz value (default when <= 0: 1e-10); the TRUE residuals |H u - lambda u| are returned
 *   cheb_order    order p >= 1 of the Chebyshev polynomial T_p (p = 1: plain Lanczos on -H); default when 0: 24
 *   cheb_lo/hi    the filter maps [cheb_lo, cheb_hi] to [-1, 1]: eigenvalues below cheb_lo are amplified.  cheb_hi <= 0:
 *                 1.15 x a power-iteration estimate of the largest eigenvalue; cheb_lo <= 0: cheb_hi / 10.
 *                 The window is verified after convergence: all n_ev returned eigenvalues must lie below cheb_lo (else
 *                 fewer than n_ev modes were amplified, or a mode above cheb_hi was -- an even-order T_p amplifies those
 *                 too -- and the returned pairs, though converged, would not be the lowest).  If not, the run is
 *                 repeated with cheb_lo raised / cheb_hi widened (up to 3 times; info reports the window finally used
 *                 and the total work); COLA_ENOCONV if that does not settle it.
 *   seed          of the deterministic start vector
 * Workspace: DEVICE, cola_eig_workspace_bytes(c, ep) bytes (n_kr + (n_kr + n_ev)/2 + 6 fp64 half-lattice vectors),
 * borrowed for the call.  evals_host / resid_host: HOST arrays of n_ev doubles (ascending eigenvalues, |H u - lambda u|
 * with |u| = 1); evecs_dev: DEVICE, n_ev fp64 even half-lattice internal vectors back to back, orthonormal (may be
 * NULL).  COLA_ENOCONV (results of the last restart filled in) if max_restarts is reached. */
typedef struct {
    int n_ev, n_kr;
    double tol;
    int max_restarts;       /* default when 0: 100 */
    int cheb_order;
    double cheb_lo, cheb_hi;
    unsigned seed;
} cola_eig_params;
typedef struct {
    int restarts;
    int op_applications;    /* applications of H = S^+ S (two Schur applications each) */
    double cheb_lo, cheb_hi;/* the filter window used */
    double seconds;
} cola_eig_info;
size_t cola_eig_workspace_bytes(const cola_ctx *c, const cola_eig_params *ep);
cola_status cola_eig_lowest(cola_ctx *c, const cola_eig_params *ep, void *work_dev, size_t work_bytes, double *evals_host, double *resid_host,
                            void *evecs_dev, cola_eig_info *info);
/* cola_cg_solve (CGNR, even_odd = 1) started from the deflated guess x0_e = sum_i u_i <u_i, S^+ bhat_e> / lambda_i built
 * from n_ev eigenpairs of H (cola_eig_lowest's output: evecs_dev DEVICE, evals_host HOST): the low modes that set the
 * condition number are solved exactly at the start, the iteration works on the rest.  Same result as cola_cg_solve. */
cola_status cola_cg_solve_deflated(cola_ctx *c, const cola_solve_params *sp, const void *b_canon_dev, void *x_canon_dev, cola_solve_info *info,
                                   const void *evecs_dev, const double *evals_host, int n_ev);

/* End-to-end variants: HOST canonical buffers; the host<->device copies are part of the call. */
cola_status cola_dslash_apply_host(cola_ctx *c, cola_prec prec, cola_parity out_parity, const void *in_canon_host, void *out_canon_host);
cola_status cola_fermion_matrix_apply_host(cola_ctx *c, cola_prec prec, int dagger, const void *in_canon_host, void *out_canon_host);
cola_status cola_cg_solve_host(cola_ctx *c, const cola_solve_params *sp, const void *b_canon_host, void *x_canon_host, cola_solve_info *info);

/* ---- Multi-right-hand-side operators and batched solver (BJ:c3 has 12 sources per gauge
 * field, one per spin-colour component).  The operators act on nrhs (1..16) vectors in ONE pass over the links and
 * the clover field: a thread block covers the sites of a single-rhs block for several right-hand sides, so gauge and
 * clover traffic is paid once per launch instead of once per vector (trade work for global-memory traffic).
 * Per vector the arithmetic, its order and hence the result are those of the single-rhs entry points.
 * "nrhs vectors" = nrhs internal buffers of the stated size stored back to back.
 *
 * Workspace: a second caller-owned DEVICE buffer holding, per right-hand side, the Schur temporaries (1.5 fp64
 * half-lattice vectors: enough for the cola_*_apply_mrhs operators, for_solver = 0) and, with for_solver != 0, the
 * vectors of the batched solver as well (5.5 fp64 half-lattice vectors).  cola_set_mrhs_workspace accepts either size;
 * cola_cg_solve_mrhs returns COLA_ENOTREADY on an operators-only workspace.  Borrowed until cola_destroy / the next
 * call; cola_set_mrhs_workspace(c, NULL, 0, 0) gives it back. */
size_t cola_mrhs_workspace_bytes(const cola_ctx *c, int nrhs, int for_solver);
cola_status cola_set_mrhs_workspace(cola_ctx *c, void *dev_ptr, size_t bytes, int nrhs);
/* out_p[n] = D_{p,1-p} in[n]: nrhs half-lattice internal DEVICE vectors each, no overlap. */
cola_status cola_dslash_apply_mrhs(cola_ctx *c, cola_prec prec, cola_parity out_parity, int nrhs, const void *in_dev, void *out_dev);
/* out[n] = M in[n] (M^+ if dagger): nrhs full internal DEVICE vectors each. */
cola_status cola_fermion_matrix_apply_mrhs(cola_ctx *c, cola_prec prec, int dagger, int nrhs, const void *in_full_dev, void *out_full_dev);
/* out_e[n] = S in_e[n] (S^+ if dagger): nrhs half-lattice (even) internal DEVICE vectors each. */
cola_status cola_schur_apply_mrhs(cola_ctx *c, cola_prec prec, int dagger, int nrhs, const void *in_even_dev, void *out_even_dev);
/* Batched solve of M x_n = b_n, n < nrhs, by the mixed-precision even-odd solvers (sp->even_odd = 1, sp->mixed = 1, 2 or 3;
 * sp->method COLA_CGNR or COLA_BICGSTAB): the systems advance in lock step, each with its own scalars, stopping test and
 * reliable-update schedule (SURVEY O7/O8 per system); a system that has converged drops out of the batch.  With
 * COLA_BICGSTAB the two applications of S per pass are multi-rhs launches and the vector updates are the single-system
 * BiCGStab's kernels, one system after the other.  b_canon_dev / x_canon_dev: nrhs
 * canonical complex128 DEVICE arrays back to back (b and x must not overlap; during the call x also holds the
 * solver's internal iterates, its final content is the canonical solution); infos: HOST array of nrhs entries
 * (seconds = time of the whole batch).  COLA_ENOCONV if any system hit max_iter (its info has the last residual).
 * COLA_EINVAL if BiCGStab broke down in a system: only that system leaves the batch (x = its iterate at its last
 * reliable update, info filled, converged by its true_residual or not), the others are solved as usual.  COLA_ENOTREADY without a
 * multi-rhs workspace for nrhs systems. */
cola_status cola_cg_solve_mrhs(cola_ctx *c, const cola_solve_params *sp, int nrhs, const void *b_canon_dev, void *x_canon_dev, cola_solve_info *infos);

/* ==== Measurement and tuning aids =====================================================================================
 * Not part of the method: switches and counters that bench.py and the A/B experiments of DESIGN.md section 6 use.  None of
 * them changes what an operator or solver computes (bit-identical results, except the summation order of fused norms
 * under cola_set_staging). */

/* Which kernel family the single-right-hand-side fp32 / 16-bit operators use.  0 (default; DESIGN.md section 6 says why):
 * every thread loads its 8 neighbour spinors from global memory through L1; 1: a thread block owns a 4-D tile of sites and
 * stages the tile's input spinors and its six faces in shared memory with bulk asynchronous copies, so that neighbours are
 * read with LDS (BJ:ns "shared-memory ... staging of neighbour half-spinors").  fp64 operators and lattices the tiles do
 * not fit (X > 512) use mode 0 regardless. */
cola_status cola_set_staging(cola_ctx *c, int mode);
/* bit 0: COLA_F32_R8 reads the 8-real links (else the context's fp32 links, 12 or 18 reals, i.e. it is COLA_F32); bit 1:
 * the fp32 operators (COLA_F32, COLA_F32_R8) read A in its 48-real form (else the 72-real packed blocks, which needs
 * COLA_FEAT_A72).  Default 3.  COLA_EINVAL outside 0..3. */
cola_status cola_set_compact(cola_ctx *c, int mask);
/* With enable != 0 every later launch of the fused dslash + clover + xpay kernel in fp32 / 16-bit
 * (Schur kernel 2 / M: the dominant kernel of a mixed-precision solve) is bracketed by a pair of CUDA events on the
 * context's stream, up to 4096 launches; cola_profile_result synchronises, returns the average duration in ms of the
 * launches that did work, their count and the number of speculative launches that returned at once, and clears the
 * window.  The event pairs cost about a microsecond per launch; leave it off for timed runs. */
cola_status cola_profile_kernel(cola_ctx *c, int enable);
cola_status cola_profile_result(cola_ctx *c, double *avg_ms, int *count, int *skipped);

/* Host-only self-test (no GPU, no context): the magic-number division the kernels use for site indices against the
 * hardware division, thread-block tile shapes and sweep-order permutations against their invariants.  msg (HOST, may be
 * NULL) receives "ok" or the first failure.  COLA_OK or COLA_EINVAL. */
cola_status cola_selftest_host(char *msg, size_t msg_len);

/* Measurement aid: number of kernels this context has launched since creation (bench.py's gpu_launches). */
unsigned long long cola_launch_count(const cola_ctx *c);

#ifdef __cplusplus
}
#endif
#endif /* COLA_H */
