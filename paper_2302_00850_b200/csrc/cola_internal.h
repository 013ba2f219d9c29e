// cola_internal.h -- shared declarations of the CUDA library (not part of the public ABI).
// Layouts and notation follow include/cola.h and DESIGN.md.  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>
#include <string.h>

#include "../../include/cola.h"

namespace cola {

// Lattice geometry as the kernels see it.  Checkerboard ("cb") index of a site of either parity:
//   cb = (x >> 1) + Xh*(y + Y*(z + Z*t)),  x = 2*(cb % Xh) + ((y + z + t + parity) & 1)
// Division of a site index n < 2^31 by a run-time extent d without the hardware's ~30-instruction
// integer-division sequence: floor(n/d) = umulhi(n, m) >> sh with m = ceil(2^(32+sh)/d), sh = ceil(log2 d) - 1
// (exact for n < 2^31 because m*d - 2^(32+sh) < d <= 2^(sh+1)); d = 1 is the identity.
struct FastDiv {
    unsigned d, m, sh;
#ifdef __CUDACC__
    __device__ __forceinline__ unsigned div(unsigned n) const { return d == 1u ? n : (__umulhi(n, m) >> sh); }
#endif
};
inline FastDiv make_fastdiv(unsigned d)
{
    FastDiv f = {d, 0u, 0u};
    if (d <= 1u) return f;
    unsigned L = 0;
    while ((1ull << L) < d) L++;
    f.sh = L - 1;
    f.m = (unsigned)((((unsigned long long)1 << (31 + L)) + d - 1) / d);
    return f;
}

struct Geom {
    int X, Y, Z, T;   // extents
    int Xh;           // X/2
    int Vh;           // half volume
    int bc[4];        // +1 / -1
    FastDiv dXh, dY, dZ;   // index decomposition of the dslash kernels
};

// Bytes of one link per site in each storage format.
// LINK_I16_12: rows 1 and 2 as 16-bit fixed point (x 32767), 24 bytes per link = one 16-byte and
// one 8-byte chunk; it comes with the fp16 clover field (CLOVER_H16_BYTES per site) and fp32 spinors and arithmetic.
// LINK_F32_8 (COLA_F32_R8): 8 fp32 reals per link = two 16-byte chunks
//   [Re U01, Im U01, Re U02, Im U02 | Re b1, Im b1, arg(U00)/pi, arg(c1)/pi],
// (b1, c1) = (U10, U20), or (U20, -U10) when |U10| > |U20| (flag = mantissa LSB of the second angle), so that
// |c1|^2 = 1 - |U00|^2 - |b1|^2 is formed without cancellation; the rest of rows 2 and 3 follows from unitarity and
// det U = 1 (reconstruct8 in cola_device.cuh).  |U00| = sqrt(1 - |U01|^2 - |U02|^2) is ill-conditioned for |U00| -> 0 (absolute
// error ~ eps/(2 |U00|), sqrt(eps) at worst): the upload measures min |U00|^2 and offers the format only if it is >= R8_MIN_U00SQ.
// Links with U01 = U02 = 0 (block diagonal, e.g. the unit matrix) are
// not covered by that parametrisation: they are flagged (mantissa LSB of the first angle) and store U11, U12 instead.
enum LinkFmt { LINK_F64_18 = 0, LINK_F32_18 = 1, LINK_F32_12 = 2, LINK_I16_12 = 3, LINK_F32_8 = 4 };
__host__ __device__ inline size_t link_bytes(int fmt)
{
    return fmt == LINK_F64_18 ? 144 : (fmt == LINK_F32_18 ? 72 : (fmt == LINK_F32_12 ? 48 : (fmt == LINK_F32_8 ? 32 : 24)));
}
constexpr double R8_MIN_U00SQ = 0.01;
constexpr size_t CLOVER_H16_BYTES = 144;   // 2 blocks x (4 x 16 B + 1 x 8 B) = 72 halfs
// 48-real form of A (SURVEY 8(f) NEXT-2 "rebuilding A from the 48-real field strength in-kernel"): per chiral block the
// three traceless Hermitian 3x3 matrices G_j = -kappa*csw*B_j of  block = 1 + [[G3, G1 - i G2], [G1 + i G2, -G3]]
// (B_j: the field-strength combinations in cola_clover.cu), each as [d0, d1, Re l10, Im l10 | Re l20, Im l20, Re l21, Im l21]
// (d2 = -d0 - d1), order G3, G1, G2: 24 reals per block, [block][chunk][Vh].  Needs trace_sub (traceless F).
constexpr size_t CLOVER_G48_REALS = 48;

// Device-resident scalars of the CG recurrence (all reductions land here; alpha and beta are
// formed inside the consuming kernels, so the host only ever reads `rr`).
struct Ctl {
    double gam[2];     // |s_k|^2 in gam[k & 1], |s_{k+1}|^2 in gam[(k + 1) & 1]
    double qq;         // |K p|^2
    double rr;         // |r|^2
    double aux[4];
    // decision state of the iteration (written by r_update's last block, read by the host with a lag)
    double rmax2;      // max |r|^2 since the last reliable update
    double target2;    // (tol |b|)^2
    double delta2;     // delta^2 of the reliable-update test; 0 = pure-precision solve
    int flag;          // 1: iteration `iters` converged or asked for a reliable update -> later kernels skip
    int iters;         // CGLS passes completed
    unsigned counter[8];  // "last block" tickets, one per concurrently used reduction
};

// Device-resident scalars of BiCGStab, complex as (re, im).  rho = <rhat, r_{i-1}> of the running
// pass, rho_next = <rhat, r_i> (formed by the x/r update or, after a reliable update, by a dot kernel), beta for the
// next search direction.  The decision state mirrors Ctl's.
struct CtlB {
    double rho[2], rho_next[2], rv[2], ts[2], beta[2];
    double tt;          // |t|^2 (fused into the operator kernel)
    double rr;          // |r|^2
    double rmax2, target2, delta2;
    int flag, iters;
    unsigned counter[4];
};

constexpr int MRHS_MAX = 16;   // right-hand sides per batched launch / solve

// Device-resident scalars of the batched (multi-right-hand-side) CGLS: one entry per vector.  Lives in the control
// block next to Ctl.  `flag` stops the whole batch (every queued kernel becomes a no-op) when any active system asks
// for a reliable update or converges; `trig` says which ones.
struct CtlM {
    double gam[2][MRHS_MAX];
    double qq[MRHS_MAX];
    double rr[MRHS_MAX];
    double rmax2[MRHS_MAX];
    double target2[MRHS_MAX];
    double delta2;
    int flag;
    int iters;
    unsigned trig;        // bit n: vector n raised the flag in iteration `iters`
};
// What the decision kernel publishes into mapped pinned host memory (rr, trig, flag first; `iters` last, after a
// system fence: it is the sequence number the host polls).
struct HostStatusM {
    double rr[MRHS_MAX];
    unsigned trig;
    int flag;
    int iters;
};
struct MrhsList { int v[MRHS_MAX]; };

// Record `msg` as this thread's context-free error message (returned by cola_last_error(NULL)).  Defined in cola_api.cu.
void set_thread_error(const char *msg);

constexpr unsigned REDUCE_GROUP = 256;
__host__ __device__ inline size_t reduce_groups(size_t nblocks) { return (nblocks + REDUCE_GROUP - 1) / REDUCE_GROUP; }

// Buffers of one deterministic grid-wide reduction (see grid_sum_last in cola_device.cuh)
constexpr int REDUCE_MAXC = 4;   // values a single launch may reduce at once (BiCGStab: |r|^2 and a complex dot)
struct ReduceWs {
    double *partials;     // [REDUCE_MAXC][pstride]: per-block partials of component c at partials + c*pstride
    double *gpart;        // [REDUCE_MAXC][gstride]
    unsigned *gticket;    // [max groups], zero before first use, self-resetting
    unsigned pstride, gstride;
};

// What r_update's last block publishes for the host: written straight into mapped pinned host memory
// (rr and flag first, then a system fence, then `iters` as the sequence number the host polls).
struct HostStatus {
    double rr;
    int flag;
    int iters;
};

// Arguments of the fused parity-dslash kernel family:
//   v   = D_{p,1-p} in                                (hopping term)
//   v   = Cy*y + coef*v        if y      (Cy = A_p if clov_y else 1)     (H6/H7/H8 epilogue)
//   v   = Cpost*v              if clov_post                              (H6: A^-1)
//   out = v;  *norm_out = sum |v|^2 if partials                          (H9)
// Sweep order of the thread blocks over the lattice.  A neighbour spinor is used three times one time slice apart
// (hops from t-1, from its own slice, from t+1); L2 serves the second and third use only if the reused spinors of three
// slices fit beside the streaming data.  When they do not (fp64 at 64^3x128, many right-hand sides), the blocks sweep
// the lattice in bands of `zb` z-planes: all time slices of one band before the next band, so the reuse distance
// shrinks to one band-slice at the price of re-reading the two z-planes next to each band.  `on == 0`: linear order.
struct Sweep {
    int on;
    int zb;            // z-planes (single-rhs) or z-tiles (multi-rhs) per band
    FastDiv d_up;      // block units per z-plane (single-rhs: Xh*Y/64) or tiles along x*y ... see the kernels
    FastDiv d_zb;
    FastDiv d_t;       // time extent (in tiles for the multi-rhs kernels)
};
// zb = 0 (off) if three slices of `bytes_per_site` reused bytes fit `l2_budget`, else the largest divisor of nz
// (a multiple of `mult`) whose three band-slices fit, at least `mult`
int choose_zband(int sites_per_plane, int nz, size_t bytes_per_site, size_t l2_budget, int mult);

struct DslashArgs {
    Geom g;
    Sweep sweep;            // single-rhs kernels; needs (Xh*Y) % 64 == 0
    const void *in;         // parity 1-p, internal half spinor
    void *out;              // parity p
    const void *gauge_p;    // links of parity p:   [mu][chunk][Vh]
    const void *gauge_q;    // links of parity 1-p
    const void *y;          // parity p half spinor or nullptr
    const void *clov_y;     // packed clover of parity p or nullptr
    int clov_y_g48;         // clov_y is the 48-real field-strength form (CLOVER_G48_REALS), expanded in the kernel
    const void *clov_post;  // packed clover applied to the result or nullptr
    double coef;
    double sgn;             // -1: D (forward hop projects with 1 - gamma_mu); +1: gamma_5 D gamma_5
    int parity;             // p
    ReduceWs red;           // reduction buffers (red.partials == nullptr: no norm)
    unsigned *counter;
    double *norm_out;
    double *dot_out;        // with norm_out and y: dot_out[0..1] = sum conj(out) * y (complex), reduced together with the norm
    int norm_accumulate;    // 1: *norm_out += sum (second half of a full-lattice operator)
    const int *skip;        // if non-null and *skip != 0 the launch is a no-op (speculatively queued iteration)
};

// Shared-memory-staged variant of the kernel family (cola_dslash_tile.cu): a block owns the 4-D tile Xh x TY x TZ x TT
// of output sites and stages the tile's input spinors plus its six faces (nent spinors) in shared memory.
struct TileShape {
    int ok;
    int TY, TZ, TT;
    int nthr;     // sites (threads) per tile
    int nent;     // staged input spinors per tile
};
TileShape choose_tile(const Geom &g);
struct TileArgs {
    DslashArgs d;          // d.sweep is ignored (tiles are swept y, z, t)
    int TX, TY, TZ, TT;
    int nthr, nent, ntiles;
    int stride;            // shared-memory entries per 16-byte chunk plane
    int off_z, off_t;      // first entry of the z faces (z-, z+) and of the t faces (t-, t+); y faces are rows of the main block
    FastDiv dTX, dTY, dTZ, d1;
    FastDiv nby, nbz;      // tiles along y and z
};
// cudaErrorNotSupported if the format or the geometry has no staged kernel (the caller falls back to launch_dslash)
cudaError_t launch_dslash_tile(int fmt, const DslashArgs &a, cudaStream_t s);

// Multi-right-hand-side launch of the same kernel family: `nrhs` vectors share one pass over
// the links and the clover field.  Vector k of the launch is vector list[k] of the caller's arrays: `in`, `out`, `y`
// of `d` point at vector 0 and consecutive vectors are `*_stride` bytes apart.  A thread block covers the sites of a
// single-rhs block for MRHS_PER_BLOCK right-hand sides (threadIdx.y), so the link a site needs is fetched from L2
// once per block and served to the other right-hand sides by L1; blocks of the same sites and different rhs groups
// are adjacent in the grid, so DRAM sees each link once per launch.
// 4-D tile of sites covered by one thread block of the multi-rhs kernels: 2^sh[0] x 2^sh[1] x 2^sh[2] x 2^sh[3]
// (x in checkerboard sites), each extent dividing the lattice extent.  With several right-hand sides per link the
// kernels are bound by L2-to-L1 traffic, most of it neighbour spinors; a compact tile lets L1 serve the neighbours
// inside the tile in all four directions (the single-rhs kernels are DRAM-bound and prefer long contiguous runs).
struct Tile {
    int sh[4];
    int vol;          // sites per tile
    int ntiles;
    FastDiv nb[3];    // tiles along x, y, z
};
Tile make_tile(const Geom &g, int max_sites, int max_x);

struct MrhsArgs {
    DslashArgs d;           // d.sweep.zb = z-PLANES per band wanted (0: linear); the launcher converts it to tiles
    Tile tile;
    Sweep tsweep;           // the same in units of tiles (filled by the launcher)           // d.red / d.counter / d.norm_out unused (per-rhs norms go through `partials`)
    int nrhs;               // right-hand sides of this launch, 1..MRHS_MAX
    int ngroups;            // rhs groups per site block (filled by the launcher)
    int nsb;                // site blocks (filled by the launcher)
    size_t in_stride, out_stride, y_stride;
    int list[MRHS_MAX];
    double *partials;       // [vector][nsb] per-block |v|^2, or nullptr; reduce with launch_mrhs_reduce
};

// launchers (cola_dslash.cu)
cudaError_t launch_dslash_mrhs(int fmt, MrhsArgs &m, cudaStream_t s);
int mrhs_tile_z(const Geom &g);        // z extent of the multi-rhs tile (bands are whole tiles)
int mrhs_site_blocks(const Geom &g);   // site blocks (tiles) of a multi-rhs launch = partial sums per vector
// out[list[k]] (+)= sum_sb partials[list[k]*nsb + sb], fixed order
cudaError_t launch_mrhs_reduce(const double *partials, int nsb, int nrhs, const int *list, double *out, int accumulate, const int *skip, cudaStream_t s);
size_t dslash_grid_blocks(size_t Vh);   // blocks a dslash launch uses = partial sums it may write
cudaError_t launch_dslash(int fmt, const DslashArgs &a, cudaStream_t s);
Sweep make_sweep(const Geom &g, int zb);   // single-rhs sweep descriptor for bands of zb z-planes (zb = 0 or unsuitable geometry: off)
// clover-only apply: out = C in on one parity (cola_dslash.cu)
cudaError_t launch_clover_apply(cola_prec prec, const Geom &g, const void *clov, const void *in, void *out, cudaStream_t s);

// layout / setup kernels (cola_layout.cu, cola_clover.cu)
cudaError_t launch_gauge_reorder(const Geom &g, const double *canon_dev, long site_lo, long n_sites, void *gauge64, void *gauge32,
                                 int fmt32, void *gauge16, void *gauge8, unsigned long long *max_dev_bits, unsigned long long *min_u00_bits, cudaStream_t s);
cudaError_t launch_spinor_pack(cola_prec prec, const Geom &g, const void *canon, void *internal, cudaStream_t s);
cudaError_t launch_spinor_unpack(cola_prec prec, const Geom &g, const void *internal, void *canon, cudaStream_t s);
cudaError_t launch_spinor_convert(cola_prec dst_prec, const void *src, void *dst, size_t n_sites, cudaStream_t s);
// a32_parities: 2 = fp32 copy of A on both parities, 1 = even parity only (no COLA_FEAT_FULL_M)
// clovG32: 48-real fp32 form of A on a32_parities parities, or nullptr
cudaError_t launch_clover_build(const Geom &g, const void *gauge64, double kappa_csw, int trace_sub, void *clovA64, void *clovA32, int a32_parities, void *clovA16,
                                void *clovG32, cudaStream_t s);
// *min_pivot_key (device, initialised to ~0ull) receives the order-preserving key of the smallest Gauss-Jordan pivot: decode with pivot_from_key
cudaError_t launch_clover_invert(const Geom &g, const void *clovA64_odd, void *clovI64, void *clovI32, void *clovI16, unsigned long long *min_pivot_key, cudaStream_t s);
inline double pivot_from_key(unsigned long long k)
{
    const unsigned long long b = (k >> 63) ? (k & 0x7fffffffffffffffull) : ~k;
    double v;
    memcpy(&v, &b, sizeof(v));
    return v;
}
cudaError_t launch_clover_unpack(const Geom &g, const void *clov64, int parity_mask, void *canon, cudaStream_t s);

// fused BLAS-1 (cola_blas.cu).  n = number of sites of the vectors (Vh or V).
int blas_max_blocks();
cudaError_t launch_norm2(cola_prec prec, const void *v, size_t n_sites, const ReduceWs &red, unsigned *counter, double *out, cudaStream_t s);
// cur = k & 1.  r -= alpha q with alpha = ctl->gam[cur] / ctl->qq;  ctl->rr = |r|^2
// and the stop / reliable-update decision: ctl->iters = iter; ctl->flag = 1 if |r|^2 <= target2 or < delta2*rmax2
cudaError_t launch_r_update(cola_prec prec, void *r, const void *q, Ctl *ctl, int cur, int iter, const int *skip, HostStatus *mirror, size_t n_sites, const ReduceWs &red, cudaStream_t s);
// x += alpha p (if do_x);  p = s + beta p with beta = gam[cur^1]/gam[cur] (if do_p)
cudaError_t launch_xp_update(cola_prec prec, void *x, void *p, const void *sv, const Ctl *ctl, int cur, int do_x, int do_p, const int *skip, size_t n_sites, cudaStream_t s);
// out64 = a*A64 + b*B64 (+ optional fp32 copy of the result, + optional |out|^2)
cudaError_t launch_axpby64(void *out64, double a, const void *A64, double b, const void *B64, void *out32, size_t n_sites,
                           const ReduceWs *red, unsigned *counter, double *norm_out, cudaStream_t s);
// x64 += x32; x32 = 0
cudaError_t launch_accumulate(void *x64, void *x32, size_t n_sites, cudaStream_t s);

// ---- BiCGStab BLAS-1 (cola_blas.cu).  Vectors are n_sites half- or full-lattice spinors of precision prec.
// which = 0: ctl->rv = <a, b>, and ctl->rho = ctl->rho_next (a new pass starts);  1: ctl->ts = <a, b>;
// 2: ctl->rho_next = <a, b> and beta = (rho_next / rho)(alpha / omega) (after a reliable update replaced r)
cudaError_t launch_bicg_dot(cola_prec prec, const void *a, const void *b, CtlB *ctl, int which, const int *skip, size_t n_sites, const ReduceWs &red, cudaStream_t s);
// s = r - alpha v, alpha = rho / rv
cudaError_t launch_bicg_s_update(cola_prec prec, void *sv, const void *r, const void *v, const CtlB *ctl, const int *skip, size_t n_sites, cudaStream_t s);
// x += alpha p + omega s;  r = s - omega t, omega = ts / tt;  ctl->rr = |r|^2, rho_next = <rhat, r>, beta; decision + status
cudaError_t launch_bicg_xr_update(cola_prec prec, void *x, void *r, const void *p, const void *sv, const void *t, const void *rhat, CtlB *ctl, int iter,
                                  const int *skip, HostStatus *mirror, size_t n_sites, const ReduceWs &red, cudaStream_t s);
// p = r + beta (p - omega v)
cudaError_t launch_bicg_p_update(cola_prec prec, void *p, const void *r, const void *v, const CtlB *ctl, const int *skip, size_t n_sites, cudaStream_t s);

// ---- low-mode solver (cola_eig.cu): fp64 half-lattice vectors of n_sites sites
cudaError_t launch_eig_cdot(const void *a, const void *b, size_t n_sites, const ReduceWs &red, unsigned *counter, double *out2, cudaStream_t s);   // out2 = <a, b>
cudaError_t launch_eig_caxpy(void *w, const void *v, size_t n_sites, const double *coef2, double scale, cudaStream_t s);                     // w += scale * coef2 * v
cudaError_t launch_eig_normalise(void *out, const void *in, size_t n_sites, const double *norm2, cudaStream_t s);                           // out = in / sqrt(norm2[0])
cudaError_t launch_eig_lincomb(void *out, double a, const void *x, double b, const void *y, double c, const void *z, size_t n_sites, cudaStream_t s);
// out[q] = sum_j V[j] Y[j][q] (j < m, q < kq; vectors vec_bytes apart; Y row-major m x kq on the device; out must not overlap V)
cudaError_t launch_eig_rotate(void *out, const void *V, size_t vec_bytes, int m, int kq, const double *Y_dev, size_t n_sites, cudaStream_t s);
cudaError_t launch_eig_start(void *v, size_t n_sites, unsigned long long seed, cudaStream_t s);
void jacobi_eigh(int m, double *A, double *w, double *Q);   // host: real symmetric A (destroyed) -> ascending w, eigenvectors in the columns of Q

// ---- batched BLAS-1 over the vectors list.v[0..nrhs) (cola_blas.cu); vector n of an array starts n*stride bytes in.
int blas_mrhs_blocks(size_t n_sites, cola_prec prec);   // blocks per vector of a batched BLAS launch = partials per vector
// r[n] -= alpha_n q[n], alpha_n = gam[cur][n]/qq[n];  partials[n][block] = block sums of |r[n]|^2
cudaError_t launch_r_update_mrhs(cola_prec prec, void *r, const void *q, size_t stride, const CtlM *ctl, int cur, const MrhsList &list, int nrhs,
                                 const int *skip, size_t n_sites, double *partials, cudaStream_t s);
// after launch_mrhs_reduce(partials -> ctl->rr): rmax2, per-vector trigger, ctl->flag, status -> mapped host memory
cudaError_t launch_decide_mrhs(CtlM *ctl, const MrhsList &list, int nrhs, int iter, const int *skip, HostStatusM *mirror, cudaStream_t s);
// x[n] += alpha_n p[n] (do_x);  p[n] = s[n] + beta_n p[n], beta_n = gam[cur^1][n]/gam[cur][n] (do_p)
cudaError_t launch_xp_update_mrhs(cola_prec prec, void *x, void *p, const void *sv, size_t stride, const CtlM *ctl, int cur, const MrhsList &list, int nrhs,
                                  int do_x, int do_p, const int *skip, size_t n_sites, cudaStream_t s);

}  // namespace cola
