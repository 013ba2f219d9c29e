// cola_dslash.cu -- the parity dslash kernel family (BJ:ns).
//
// One thread per output site ("each lattice site is mapped to a single thread").  For each of
// the 8 hops: load the neighbour spinor (SoA, 16-byte chunks, site index fastest => coalesced),
// spin-project it to a half spinor BEFORE the colour multiply (12 instead of 24 reals through the
// SU(3) mat-vec), load the link (12 reals + in-register third-row reconstruction, or 18), multiply,
// apply the boundary sign, reconstruct the lower spin components and accumulate.  The clover
// mat-vec, the xpay and the |.|^2 reduction are epilogues of the same kernel, so a Schur-complement
// application is two launches and no intermediate vector is re-read for BLAS-1 work.
//
// Chiral basis: gamma_mu = [[0, A_mu], [A_mu^+, 0]], A_k = -i sigma_k, A_t = 1:
//   (1 + s gamma_mu) psi = [ h ; s A_mu^+ h ],   h = psi_upper + s A_mu psi_lower,   s = +-1.
#include <string.h>

#include "cola_hop.cuh"

namespace cola {

namespace {

// Tuning knobs (compile-time).  Defaults = best of the round-1 sweeps on B200: 64 threads per
// block; fp32 kernels software-pipelined two hops ahead with 128 registers (8 blocks = 16 warps per SM);
// fp64 kernels unpipelined at 168 registers (6 blocks = 12 warps per SM).  Without pipelining the best fp32 point was
// 80 registers (12 blocks): the kernels are bound by bytes in flight, which either more warps or loads issued ahead of
// use provide; two hops ahead at 16 warps beats 24 warps without by 5-9 % (one hop ahead: 4-8 %).
#ifndef COLA_DSLASH_BLOCK
#define COLA_DSLASH_BLOCK 64
#endif
#ifndef COLA_DSLASH_MINB_F32
#define COLA_DSLASH_MINB_F32 8
#endif
#ifndef COLA_DSLASH_MINB_F64
#define COLA_DSLASH_MINB_F64 6
#endif
constexpr int DSLASH_BLOCK = COLA_DSLASH_BLOCK;
template <int FMT> struct MinBlocks { static constexpr int value = (FMT == LINK_F64_18) ? COLA_DSLASH_MINB_F64 : COLA_DSLASH_MINB_F32; };

// one hop: neighbour index nb (parity 1-p), link at site li of the given gauge block
template <int FMT, int MU, bool BACK, bool STREAM, typename T>
__device__ __forceinline__ void hop(const void *in, const char *gauge_mu, size_t Vh, int nb, int li, T eta, T s, T (&acc)[24])
{
    T psi[24], h[12], g[12], u[18];
    load_reals<T, 24, false>(in, Vh, nb, psi);
    load_link<FMT, STREAM>(gauge_mu, Vh, li, u);
    project<MU>(psi, s, h);
    su3_mul<BACK>(u, h, g);
    reconstruct_accumulate<MU>(g, eta, s, acc);
}

// Hop H = 2*MU + BACK of the pipelined sequence: consumes (psi, raw) of hop H, then refills them with hop H+1's
// neighbour spinor `nb_next` and link `li_next` of `gauge_next` (nullptr: last hop).
template <int FMT, int H, bool STREAM, int LAST_REFILL = 7, typename T>
__device__ __forceinline__ void hop_pipe(const void *in, const char *gauge_next, size_t Vh, int nb_next, int li_next, T (&psi)[24], RawLink<FMT> &raw,
                                         T eta, T s, T (&acc)[24])
{
    constexpr int MU = H >> 1;
    constexpr bool BACK = (H & 1) != 0;
    T h[12], g[12], u[18];
    project<MU>(psi, s, h);
    expand_link<FMT>(raw, u);
    if (H < LAST_REFILL) {
        load_reals<T, 24, false>(in, Vh, nb_next, psi);
        load_raw_link<FMT, STREAM>(gauge_next, Vh, li_next, raw);
    }
    su3_mul<BACK>(u, h, g);
    reconstruct_accumulate<MU>(g, eta, s, acc);
}

// One output site i of parity a.parity:  v = D in;  v = [A] y + coef v (XPAY);  v = Cpost v (POST);  out = v.
// Returns |v|^2 if want_norm.  XPAY: 0 none, 1 v = y + coef v, 2 v = A y + coef v.   POST: 0 none, 1 v = Cpost v.
// STREAM: links and clover are read once (no L1 allocation); !STREAM: they are shared by the right-hand sides of a block.
// PDLW (16-bit kernels only): the kernel was launched as a programmatic dependent and has not waited for its predecessor
// yet: the index arithmetic and the raw links of the first two hops run before pdl_wait(); a raised skip flag
// (grid-uniform) is reported by returning -1.  (+2 % for the SM-bound 16-bit kernels; the fp32 kernels lose 1.7 % with
// the reordered first loads and wait at the top of the kernel instead.)
template <int FMT, int XPAY, int POST, bool STREAM, bool PDLW = false, bool DOT = false>
__device__ __forceinline__ double dslash_site(const DslashArgs &a, const int i, const void *in, const void *yin, void *out, const bool want_norm,
                                              double *dot = nullptr)
{
    typedef typename LinkT<FMT>::T T;
    const Geom &g = a.g;
    const size_t Vh = g.Vh;
    double nrm = 0.0;
    {
        // coordinates of the output site
        const unsigned r1 = g.dXh.div((unsigned)i), r2 = g.dY.div(r1), r3 = g.dZ.div(r2);
        const int xh = i - (int)r1 * g.Xh, y = (int)r1 - (int)r2 * g.Y, z = (int)r2 - (int)r3 * g.Z, t = (int)r3;
        const int odd = (y + z + t + a.parity) & 1;     // x = 2*xh + odd
        const int sY = g.Xh, sZ = g.Xh * g.Y, sT = g.Xh * g.Y * g.Z;

        // neighbour cb indices (parity 1-p) and boundary crossings
        const int xf = odd ? (xh + 1 == g.Xh ? i - xh : i + 1) : i;
        const int xb = odd ? i : (xh == 0 ? i + g.Xh - 1 : i - 1);
        const bool cxf = odd && (xh + 1 == g.Xh), cxb = !odd && (xh == 0);
        const int yf = (y + 1 == g.Y) ? i - (g.Y - 1) * sY : i + sY;
        const int yb = (y == 0) ? i + (g.Y - 1) * sY : i - sY;
        const int zf = (z + 1 == g.Z) ? i - (g.Z - 1) * sZ : i + sZ;
        const int zb = (z == 0) ? i + (g.Z - 1) * sZ : i - sZ;
        const int tf = (t + 1 == g.T) ? i - (g.T - 1) * sT : i + sT;
        const int tb = (t == 0) ? i + (g.T - 1) * sT : i - sT;

        const T one = 1;
        const T ex_f = (cxf && g.bc[0] < 0) ? -one : one, ex_b = (cxb && g.bc[0] < 0) ? -one : one;
        const T ey_f = (y + 1 == g.Y && g.bc[1] < 0) ? -one : one, ey_b = (y == 0 && g.bc[1] < 0) ? -one : one;
        const T ez_f = (z + 1 == g.Z && g.bc[2] < 0) ? -one : one, ez_b = (z == 0 && g.bc[2] < 0) ? -one : one;
        const T et_f = (t + 1 == g.T && g.bc[3] < 0) ? -one : one, et_b = (t == 0 && g.bc[3] < 0) ? -one : one;

        const T sf = (T)a.sgn, sb = -(T)a.sgn;   // forward: (1 + sgn*gamma), backward: (1 - sgn*gamma)
        const size_t lb = link_bytes(FMT) * Vh;  // bytes of one (parity, mu) block
        const char *gp = reinterpret_cast<const char *>(a.gauge_p);
        const char *gq = reinterpret_cast<const char *>(a.gauge_q);

        T acc[24];
#pragma unroll
        for (int k = 0; k < 24; k++) acc[k] = 0;

        if constexpr (FMT != LINK_F64_18) {
            // software-pipelined hops: the loads of hop h+2 (neighbour spinor and raw link) are issued right after the
            // projection of hop h, whose spinor registers are dead by then, so they are in flight during the SU(3)
            // multiplies and accumulations of hops h and h+1.  (Hop by hop, one hop ahead and a shared-memory FIFO
            // fed by asynchronous copies were measured and dropped: profiles/r3_experiments.md.)
            {
            // two hops ahead: buffers A (even hops) and B (odd hops); hop h refills its buffer with hop h+2
            T psiA[24], psiB[24];
            RawLink<FMT> rawA, rawB;
            if (PDLW) {
                load_raw_link<FMT, STREAM>(gp + 0 * lb, Vh, i, rawA);
                load_raw_link<FMT, STREAM>(gq + 0 * lb, Vh, xb, rawB);
                pdl_wait();
                if (a.skip && *a.skip) return -1.0;
                load_reals<T, 24, false>(in, Vh, xf, psiA);
                load_reals<T, 24, false>(in, Vh, xb, psiB);
            } else {
                load_reals<T, 24, false>(in, Vh, xf, psiA);
                load_raw_link<FMT, STREAM>(gp + 0 * lb, Vh, i, rawA);
                load_reals<T, 24, false>(in, Vh, xb, psiB);
                load_raw_link<FMT, STREAM>(gq + 0 * lb, Vh, xb, rawB);
            }
            hop_pipe<FMT, 0, STREAM, 6>(in, gp + 1 * lb, Vh, yf, i, psiA, rawA, ex_f, sf, acc);
            hop_pipe<FMT, 1, STREAM, 6>(in, gq + 1 * lb, Vh, yb, yb, psiB, rawB, ex_b, sb, acc);
            hop_pipe<FMT, 2, STREAM, 6>(in, gp + 2 * lb, Vh, zf, i, psiA, rawA, ey_f, sf, acc);
            hop_pipe<FMT, 3, STREAM, 6>(in, gq + 2 * lb, Vh, zb, zb, psiB, rawB, ey_b, sb, acc);
            hop_pipe<FMT, 4, STREAM, 6>(in, gp + 3 * lb, Vh, tf, i, psiA, rawA, ez_f, sf, acc);
            hop_pipe<FMT, 5, STREAM, 6>(in, gq + 3 * lb, Vh, tb, tb, psiB, rawB, ez_b, sb, acc);
            hop_pipe<FMT, 6, STREAM, 6>(in, nullptr, Vh, 0, 0, psiA, rawA, et_f, sf, acc);
            hop_pipe<FMT, 7, STREAM, 6>(in, nullptr, Vh, 0, 0, psiB, rawB, et_b, sb, acc);
            }
        } else
        {
        hop<FMT, 0, false, STREAM>(in, gp + 0 * lb, Vh, xf, i, ex_f, sf, acc);
        hop<FMT, 0, true, STREAM>(in, gq + 0 * lb, Vh, xb, xb, ex_b, sb, acc);
        hop<FMT, 1, false, STREAM>(in, gp + 1 * lb, Vh, yf, i, ey_f, sf, acc);
        hop<FMT, 1, true, STREAM>(in, gq + 1 * lb, Vh, yb, yb, ey_b, sb, acc);
        hop<FMT, 2, false, STREAM>(in, gp + 2 * lb, Vh, zf, i, ez_f, sf, acc);
        hop<FMT, 2, true, STREAM>(in, gq + 2 * lb, Vh, zb, zb, ez_b, sb, acc);
        hop<FMT, 3, false, STREAM>(in, gp + 3 * lb, Vh, tf, i, et_f, sf, acc);
        hop<FMT, 3, true, STREAM>(in, gq + 3 * lb, Vh, tb, tb, et_b, sb, acc);
        }

        nrm = dslash_epilogue<FMT, XPAY, POST, STREAM, DOT>(a, i, acc, yin, out, want_norm, dot);
    }
    return nrm;
}

// ---- R right-hand sides per thread (register blocking): the thread of output site i applies each
// link, loaded, converted and completed ONCE, to the spin-projected neighbours of R vectors, and each clover block, loaded
// once, to R spinors.  Per vector the arithmetic is the same sequence of calls as in dslash_site (results bit-identical,
// tested); what is shared is everything that does not depend on the vector: index arithmetic, boundary signs, 8 link
// loads + reconstructions, 2-4 clover block loads + conversions.  in/yin/out: the R vectors' arrays (entries past
// `nvalid` alias a valid vector: computed, not stored).
// Pipelining: one spinor buffer per vector, refilled with the next hop's neighbour right after the projection that
// consumed it; two raw-link buffers alternate between hops, refilled two hops ahead.
template <int FMT, int H, int R, bool STREAM, typename T>
__device__ __forceinline__ void hop_r(const char *const (&in)[R], const char *gauge_next2, size_t Vh, int nb_next, int li_next2, T (&psi)[R][24],
                                      RawLink<FMT> &raw, T eta, T s, T (&acc)[R][24])
{
    constexpr int MU = H >> 1;
    constexpr bool BACK = (H & 1) != 0;
    T u[18];
    expand_link<FMT>(raw, u);
    if (H < 6) load_raw_link<FMT, STREAM>(gauge_next2, Vh, li_next2, raw);   // the link of hop H + 2
#pragma unroll
    for (int r = 0; r < R; r++) {
        T h[12], g[12];
        project<MU>(psi[r], s, h);
        if (H < 7) load_reals<T, 24, false>(in[r], Vh, nb_next, psi[r]);   // vector r's neighbour of hop H + 1
        su3_mul<BACK>(u, h, g);
        reconstruct_accumulate<MU>(g, eta, s, acc[r]);
    }
}

template <int FMT, int XPAY, int POST, int R, bool STREAM>
__device__ __forceinline__ void dslash_site_r(const DslashArgs &a, const int i, const char *const (&in)[R], const char *const (&yin)[R], char *const (&out)[R],
                                              const int nvalid, const bool want_norm, double (&nrm)[R])
{
    typedef typename LinkT<FMT>::T T;
    typedef typename VT<T>::V V;
    constexpr int N = VT<T>::N;
    const Geom &g = a.g;
    const size_t Vh = g.Vh;
    const unsigned r1 = g.dXh.div((unsigned)i), r2 = g.dY.div(r1), r3 = g.dZ.div(r2);
    const int xh = i - (int)r1 * g.Xh, y = (int)r1 - (int)r2 * g.Y, z = (int)r2 - (int)r3 * g.Z, t = (int)r3;
    const int odd = (y + z + t + a.parity) & 1;
    const int sY = g.Xh, sZ = g.Xh * g.Y, sT = g.Xh * g.Y * g.Z;
    const int xf = odd ? (xh + 1 == g.Xh ? i - xh : i + 1) : i;
    const int xb = odd ? i : (xh == 0 ? i + g.Xh - 1 : i - 1);
    const bool cxf = odd && (xh + 1 == g.Xh), cxb = !odd && (xh == 0);
    const int yf = (y + 1 == g.Y) ? i - (g.Y - 1) * sY : i + sY;
    const int yb = (y == 0) ? i + (g.Y - 1) * sY : i - sY;
    const int zf = (z + 1 == g.Z) ? i - (g.Z - 1) * sZ : i + sZ;
    const int zb = (z == 0) ? i + (g.Z - 1) * sZ : i - sZ;
    const int tf = (t + 1 == g.T) ? i - (g.T - 1) * sT : i + sT;
    const int tb = (t == 0) ? i + (g.T - 1) * sT : i - sT;
    const T one = 1;
    const T ex_f = (cxf && g.bc[0] < 0) ? -one : one, ex_b = (cxb && g.bc[0] < 0) ? -one : one;
    const T ey_f = (y + 1 == g.Y && g.bc[1] < 0) ? -one : one, ey_b = (y == 0 && g.bc[1] < 0) ? -one : one;
    const T ez_f = (z + 1 == g.Z && g.bc[2] < 0) ? -one : one, ez_b = (z == 0 && g.bc[2] < 0) ? -one : one;
    const T et_f = (t + 1 == g.T && g.bc[3] < 0) ? -one : one, et_b = (t == 0 && g.bc[3] < 0) ? -one : one;
    const T sf = (T)a.sgn, sb = -(T)a.sgn;
    const size_t lb = link_bytes(FMT) * Vh;
    const char *gp = reinterpret_cast<const char *>(a.gauge_p);
    const char *gq = reinterpret_cast<const char *>(a.gauge_q);

    T acc[R][24], psi[R][24];
#pragma unroll
    for (int r = 0; r < R; r++)
#pragma unroll
        for (int k = 0; k < 24; k++) acc[r][k] = 0;
    RawLink<FMT> rawA, rawB;
    load_raw_link<FMT, STREAM>(gp + 0 * lb, Vh, i, rawA);
#pragma unroll
    for (int r = 0; r < R; r++) load_reals<T, 24, false>(in[r], Vh, xf, psi[r]);
    load_raw_link<FMT, STREAM>(gq + 0 * lb, Vh, xb, rawB);
    hop_r<FMT, 0, R, STREAM>(in, gp + 1 * lb, Vh, xb, i, psi, rawA, ex_f, sf, acc);
    hop_r<FMT, 1, R, STREAM>(in, gq + 1 * lb, Vh, yf, yb, psi, rawB, ex_b, sb, acc);
    hop_r<FMT, 2, R, STREAM>(in, gp + 2 * lb, Vh, yb, i, psi, rawA, ey_f, sf, acc);
    hop_r<FMT, 3, R, STREAM>(in, gq + 2 * lb, Vh, zf, zb, psi, rawB, ey_b, sb, acc);
    hop_r<FMT, 4, R, STREAM>(in, gp + 3 * lb, Vh, zb, i, psi, rawA, ez_f, sf, acc);
    hop_r<FMT, 5, R, STREAM>(in, gq + 3 * lb, Vh, tf, tb, psi, rawB, ez_b, sb, acc);
    hop_r<FMT, 6, R, STREAM>(in, nullptr, Vh, tb, 0, psi, rawA, et_f, sf, acc);
    hop_r<FMT, 7, R, STREAM>(in, nullptr, Vh, 0, 0, psi, rawB, et_b, sb, acc);

    // epilogues (dslash_epilogue in cola_hop.cuh, per chiral block so that a clover block is loaded once for the R vectors)
    if (XPAY != 0) {
        const T cf = (T)a.coef;
#pragma unroll
        for (int b = 0; b < 2; b++) {
            T c[36];
            if constexpr (XPAY == 3) load_clover_g48<T, STREAM>(a.clov_y, Vh, i, b, c);
            else if constexpr (XPAY == 2) load_clover_block<T, STREAM, FMT == LINK_I16_12>(a.clov_y, Vh, i, b, c);
#pragma unroll
            for (int r = 0; r < R; r++) {
                T yv[12];
                load_reals<T, 12, true>(reinterpret_cast<const V *>(yin[r]) + (size_t)b * (12 / N) * Vh, Vh, i, yv);
                if constexpr (XPAY == 1) {
#pragma unroll
                    for (int k = 0; k < 12; k++) acc[r][12 * b + k] = yv[k] + cf * acc[r][12 * b + k];
                } else {
                    T cy[12];
                    clover_block_mul(c, yv, cy);
#pragma unroll
                    for (int k = 0; k < 12; k++) acc[r][12 * b + k] = cy[k] + cf * acc[r][12 * b + k];
                }
            }
        }
    }
    if (POST != 0) {
#pragma unroll
        for (int b = 0; b < 2; b++) {
            T c[36];
            load_clover_block<T, STREAM, FMT == LINK_I16_12>(a.clov_post, Vh, i, b, c);
#pragma unroll
            for (int r = 0; r < R; r++) {
                T w[12];
                clover_block_mul(c, &acc[r][12 * b], w);
#pragma unroll
                for (int k = 0; k < 12; k++) acc[r][12 * b + k] = w[k];
            }
        }
    }
#pragma unroll
    for (int r = 0; r < R; r++) {
        if (r < nvalid) store_reals<T, 24>(out[r], Vh, i, acc[r]);
        nrm[r] = 0.0;
        if (want_norm) {
            T s2 = 0;
#pragma unroll
            for (int k = 0; k < 24; k++) s2 += acc[r][k] * acc[r][k];
            nrm[r] = (double)s2;
        }
    }
}

// Sweep position -> run of DSLASH_BLOCK consecutive sites (identity, or the z-banded order of Sweep in cola_internal.h)
__device__ __forceinline__ unsigned sweep_run(const Sweep &w, const Geom &g, unsigned pos)
{
    if (!w.on) return pos;
    const unsigned q1 = w.d_up.div(pos), u = pos - q1 * w.d_up.d;
    const unsigned q2 = w.d_zb.div(q1), zi = q1 - q2 * w.d_zb.d;
    const unsigned band = w.d_t.div(q2), t = q2 - band * w.d_t.d;
    return ((t * (unsigned)g.Z + band * w.d_zb.d + zi) * w.d_up.d) + u;
}

// DOT (XPAY != 0, POST == 0, with a norm): also reduces <out, y> into a.dot_out (BiCGStab's <t, s> for t = S s)
template <int FMT, int XPAY, int POST, bool DOT = false>
__global__ void __launch_bounds__(DSLASH_BLOCK, MinBlocks<FMT>::value) dslash_kernel(const __grid_constant__ DslashArgs a)
{
    constexpr bool LATE_WAIT = (FMT == LINK_I16_12);   // see dslash_site<.., PDLW>
    pdl_trigger();
    if (!LATE_WAIT) {
        pdl_wait();
        if (a.skip && *a.skip) return;
    }
    // which run of DSLASH_BLOCK consecutive sites this block covers: linear, or the z-banded sweep (block order =
    // [unit in plane, z in band, t, band])
    const unsigned run = sweep_run(a.sweep, a.g, blockIdx.x);
    const int i = (int)run * DSLASH_BLOCK + (int)threadIdx.x;
    const bool want_norm = a.red.partials != nullptr;
    double nrm = 0.0, dot[2] = {0.0, 0.0};
    if (i < a.g.Vh) {
        nrm = dslash_site<FMT, XPAY, POST, true, LATE_WAIT, DOT>(a, i, a.in, a.y, a.out, want_norm, dot);
    } else if (LATE_WAIT) {
        pdl_wait();
        nrm = (a.skip && *a.skip) ? -1.0 : 0.0;
    }
    if (LATE_WAIT && nrm < 0.0) return;   // skip flag raised: the same for every thread of the grid
    if constexpr (DOT) {   // |out|^2 and <out, y> in one deterministic reduction (the launcher guarantees norm_out and dot_out)
        const double v3[3] = {nrm, dot[0], dot[1]};
        double tot[3];
        if (grid_sum_last_n<3>(v3, a.red, a.counter, tot)) {
            *a.norm_out = a.norm_accumulate ? *a.norm_out + tot[0] : tot[0];
            a.dot_out[0] = tot[1];
            a.dot_out[1] = tot[2];
        }
    } else if (want_norm) grid_sum_finalize(nrm, a.red, a.counter, a.norm_out, a.norm_accumulate != 0);
}

// ---- multi-right-hand-side variant (MrhsArgs in cola_internal.h)
#ifndef COLA_MRHS_PER_BLOCK_F32
#define COLA_MRHS_PER_BLOCK_F32 2
#endif
#ifndef COLA_MRHS_PER_BLOCK_F64
#define COLA_MRHS_PER_BLOCK_F64 2
#endif
#ifndef COLA_MRHS_R
#define COLA_MRHS_R 2     // right-hand sides per thread of the fp32 / 16-bit multi-rhs kernels (dslash_site_r); fp64: 1
#endif
#ifndef COLA_MRHS_MINB_F32   // register budget: 128 (R = 1), 168 (R = 2), 255 (R >= 3) at 128 threads per block
#define COLA_MRHS_MINB_F32 (COLA_MRHS_R == 1 ? 4 : (COLA_MRHS_R == 2 ? 3 : 2))
#endif
#ifndef COLA_MRHS_MINB_F64
#define COLA_MRHS_MINB_F64 3
#endif
#ifndef COLA_MRHS_SITES
#define COLA_MRHS_SITES 64
#endif
#ifndef COLA_MRHS_TILE_X
#define COLA_MRHS_TILE_X 16
#endif
constexpr int MSITES = COLA_MRHS_SITES;
template <int FMT> struct MrhsCfg {
    static constexpr int NRB = (FMT == LINK_F64_18) ? COLA_MRHS_PER_BLOCK_F64 : COLA_MRHS_PER_BLOCK_F32;   // rows of threads (threadIdx.y)
    static constexpr int MINB = (FMT == LINK_F64_18) ? COLA_MRHS_MINB_F64 : COLA_MRHS_MINB_F32;
    static constexpr int R = (FMT == LINK_F64_18) ? 1 : COLA_MRHS_R;                                       // vectors per thread
};

template <int FMT, int XPAY, int POST>
__global__ void __launch_bounds__(MSITES * MrhsCfg<FMT>::NRB, MrhsCfg<FMT>::MINB) dslash_mrhs_kernel(const __grid_constant__ MrhsArgs m)
{
    constexpr int NRB = MrhsCfg<FMT>::NRB, R = MrhsCfg<FMT>::R;
    if (m.d.skip && *m.d.skip) return;
    const Geom &g = m.d.g;
    const Tile &tl = m.tile;
    const unsigned sb = blockIdx.x / (unsigned)m.ngroups, grp = blockIdx.x - sb * (unsigned)m.ngroups;
    const int k0 = ((int)grp * NRB + (int)threadIdx.y) * R;   // first vector of this thread
    // site of this thread: tile origin (block-uniform) + position inside the tile
    const unsigned b1 = tl.nb[0].div(sb), b2 = tl.nb[1].div(b1);
    unsigned bz, bt;
    if (m.tsweep.on) {   // z-banded sweep over tiles: [x tile, y tile, z tile in band, t tile, band]
        const unsigned q3 = m.tsweep.d_zb.div(b2), zi = b2 - q3 * m.tsweep.d_zb.d;
        const unsigned band = m.tsweep.d_t.div(q3);
        bt = q3 - band * m.tsweep.d_t.d;
        bz = band * m.tsweep.d_zb.d + zi;
    } else {
        bt = tl.nb[2].div(b2);
        bz = b2 - bt * tl.nb[2].d;
    }
    const unsigned l = threadIdx.x;
    const int s0 = tl.sh[0], s1 = tl.sh[1], s2 = tl.sh[2];
    const int xh = (int)((sb - b1 * tl.nb[0].d) << s0) + (int)(l & ((1u << s0) - 1u));
    const int y = (int)((b1 - b2 * tl.nb[1].d) << s1) + (int)((l >> s0) & ((1u << s1) - 1u));
    const int z = (int)(bz << s2) + (int)((l >> (s0 + s1)) & ((1u << s2) - 1u));
    const int t = (int)(bt << tl.sh[3]) + (int)(l >> (s0 + s1 + s2));
    const int i = xh + g.Xh * (y + g.Y * (z + g.Z * t));
    const bool want_norm = m.partials != nullptr;
    const bool live = k0 < m.nrhs && (int)l < tl.vol;
    double nrm[R];
    size_t vec[R];
#pragma unroll
    for (int r = 0; r < R; r++) {
        nrm[r] = 0.0;
        const int kr = k0 + r < m.nrhs ? k0 + r : m.nrhs - 1;   // past the end: alias the last vector (computed, not stored)
        vec[r] = (size_t)m.list[kr];
    }
    if (live) {
        if constexpr (R == 1) {
            nrm[0] = dslash_site<FMT, XPAY, POST, false>(m.d, i, reinterpret_cast<const char *>(m.d.in) + vec[0] * m.in_stride,
                                                         reinterpret_cast<const char *>(m.d.y) + vec[0] * m.y_stride,
                                                         reinterpret_cast<char *>(m.d.out) + vec[0] * m.out_stride, want_norm);
        } else {
            const char *in[R], *yin[R];
            char *out[R];
#pragma unroll
            for (int r = 0; r < R; r++) {
                in[r] = reinterpret_cast<const char *>(m.d.in) + vec[r] * m.in_stride;
                yin[r] = reinterpret_cast<const char *>(m.d.y) + vec[r] * m.y_stride;
                out[r] = reinterpret_cast<char *>(m.d.out) + vec[r] * m.out_stride;
            }
            const int nvalid = m.nrhs - k0 < R ? m.nrhs - k0 : R;
            dslash_site_r<FMT, XPAY, POST, R, NRB == 1>(m.d, i, in, yin, out, nvalid, want_norm, nrm);   // one row of threads: links and clover are read once
        }
    }
    if (want_norm) {   // one partial per (vector, site block): the warps of a row (threadIdx.y) hold R right-hand sides
        __shared__ double sm[NRB][R][MSITES / 32];
#pragma unroll
        for (int r = 0; r < R; r++) {
            const double w = warp_sum(nrm[r]);
            if ((threadIdx.x & 31) == 0) sm[threadIdx.y][r][threadIdx.x >> 5] = w;
        }
        __syncthreads();
        if (threadIdx.x < R && k0 + (int)threadIdx.x < m.nrhs) {
            double tsum = 0.0;
#pragma unroll
            for (int q = 0; q < MSITES / 32; q++) tsum += sm[threadIdx.y][threadIdx.x][q];
            m.partials[(size_t)m.list[k0 + threadIdx.x] * (size_t)m.nsb + sb] = tsum;
        }
    }
}

// out[vec] (+)= sum over site blocks of partials[vec][.], one block per right-hand side, fixed order
__global__ void __launch_bounds__(256) mrhs_reduce_kernel(const double *partials, int nsb, const __grid_constant__ MrhsList list, const int *skip, double *out, int accumulate)
{
    if (skip && *skip) return;
    __shared__ double sm[33];
    const int vec = list.v[blockIdx.x];
    const double *p = partials + (size_t)vec * nsb;
    double a = 0.0;
    for (int k = threadIdx.x; k < nsb; k += 256) a += p[k];
    a = block_sum(a, sm);
    if (threadIdx.x == 0) out[vec] = accumulate ? out[vec] + a : a;
}

template <typename T>
__global__ void __launch_bounds__(DSLASH_BLOCK) clover_apply_kernel(int Vh, const void *clov, const void *in, void *out)
{
    const int i = blockIdx.x * DSLASH_BLOCK + threadIdx.x;
    if (i >= Vh) return;
    T v[24], w[24];
    load_reals<T, 24, true>(in, Vh, i, v);
    clover_apply<T>(clov, Vh, i, v, w);
    store_reals<T, 24>(out, Vh, i, w);
}

template <int FMT>
cudaError_t launch_fmt(const DslashArgs &a, cudaStream_t s)
{
    const int xpay = a.y ? (a.clov_y ? (a.clov_y_g48 ? 3 : 2) : 1) : 0;
    const int post = a.clov_post ? 1 : 0;
    const dim3 grid((a.g.Vh + DSLASH_BLOCK - 1) / DSLASH_BLOCK), block(DSLASH_BLOCK);
    const size_t sm = 0;
    if (xpay == 0 && post == 0) launch_pdl_smem(dslash_kernel<FMT, 0, 0>, grid, block, sm, s, a);
    else if (xpay == 0 && post == 1) launch_pdl_smem(dslash_kernel<FMT, 0, 1>, grid, block, sm, s, a);
    else if (xpay == 1 && post == 0) launch_pdl_smem(dslash_kernel<FMT, 1, 0>, grid, block, sm, s, a);
    else if (xpay == 1 && post == 1) launch_pdl_smem(dslash_kernel<FMT, 1, 1>, grid, block, sm, s, a);
    else if (xpay == 2 && post == 0) {
        if (a.dot_out && a.norm_out) launch_pdl_smem(dslash_kernel<FMT, 2, 0, true>, grid, block, sm, s, a);
        else launch_pdl_smem(dslash_kernel<FMT, 2, 0>, grid, block, sm, s, a);
    } else if (xpay == 3 && post == 0) {
        if constexpr (FMT == LINK_F32_12 || FMT == LINK_F32_8 || FMT == LINK_F32_18) {
            if (a.dot_out && a.norm_out) launch_pdl_smem(dslash_kernel<FMT, 3, 0, true>, grid, block, sm, s, a);
            else launch_pdl_smem(dslash_kernel<FMT, 3, 0>, grid, block, sm, s, a);
        }
        else return cudaErrorInvalidValue;   // the 48-real form of A exists in fp32 only
    } else return cudaErrorInvalidValue;
    return cudaGetLastError();
}

template <int FMT>
cudaError_t launch_mrhs_fmt(MrhsArgs &m, cudaStream_t s)
{
    constexpr int NRB = MrhsCfg<FMT>::NRB * MrhsCfg<FMT>::R;   // vectors per block
    const int xpay = m.d.y ? (m.d.clov_y ? (m.d.clov_y_g48 ? 3 : 2) : 1) : 0;
    const int post = m.d.clov_post ? 1 : 0;
    m.tile = make_tile(m.d.g, MSITES, COLA_MRHS_TILE_X);
    m.nsb = m.tile.ntiles;
    m.ngroups = (m.nrhs + NRB - 1) / NRB;
    memset(&m.tsweep, 0, sizeof(m.tsweep));
    {
        const int tz = 1 << m.tile.sh[2], nbz = m.d.g.Z >> m.tile.sh[2], nbt = m.d.g.T >> m.tile.sh[3];
        const int zbt = m.d.sweep.zb / tz;   // band in tiles
        if (m.d.sweep.zb > 0 && zbt >= 1 && zbt < nbz && nbz % zbt == 0) {
            m.tsweep.on = 1;
            m.tsweep.zb = zbt;
            m.tsweep.d_zb = make_fastdiv((unsigned)zbt);
            m.tsweep.d_t = make_fastdiv((unsigned)nbt);
        }
    }
    const dim3 grid((unsigned)m.nsb * (unsigned)m.ngroups), block(MSITES, MrhsCfg<FMT>::NRB);
    if (xpay == 0 && post == 0) dslash_mrhs_kernel<FMT, 0, 0><<<grid, block, 0, s>>>(m);
    else if (xpay == 0 && post == 1) dslash_mrhs_kernel<FMT, 0, 1><<<grid, block, 0, s>>>(m);
    else if (xpay == 1 && post == 0) dslash_mrhs_kernel<FMT, 1, 0><<<grid, block, 0, s>>>(m);
    else if (xpay == 1 && post == 1) dslash_mrhs_kernel<FMT, 1, 1><<<grid, block, 0, s>>>(m);
    else if (xpay == 2 && post == 0) dslash_mrhs_kernel<FMT, 2, 0><<<grid, block, 0, s>>>(m);
    else if (xpay == 3 && post == 0) {
        if constexpr (FMT == LINK_F32_12 || FMT == LINK_F32_8 || FMT == LINK_F32_18) dslash_mrhs_kernel<FMT, 3, 0><<<grid, block, 0, s>>>(m);
        else return cudaErrorInvalidValue;
    } else return cudaErrorInvalidValue;
    return cudaGetLastError();
}

}  // namespace

// Tile = the largest power-of-two box of at most max_sites sites whose extents divide the lattice extents: x first, up
// to max_x checkerboard sites (coalescing), then y, z, t doubled in turn so the tile stays close to a hypercube.
Tile make_tile(const Geom &g, int max_sites, int max_x)
{
    Tile t;
    const int ext[4] = {g.Xh, g.Y, g.Z, g.T};
    int vol = 1;
    for (int k = 0; k < 4; k++) t.sh[k] = 0;
    while (vol * 2 <= max_sites && (1 << (t.sh[0] + 1)) <= max_x && ext[0] % (1 << (t.sh[0] + 1)) == 0) {
        t.sh[0]++;
        vol *= 2;
    }
    for (bool grown = true; grown && vol * 2 <= max_sites;) {
        grown = false;
        for (int k = 1; k < 4 && vol * 2 <= max_sites; k++) {
            if (ext[k] % (1 << (t.sh[k] + 1)) == 0) {
                t.sh[k]++;
                vol *= 2;
                grown = true;
            }
        }
    }
    while (vol * 2 <= max_sites && ext[0] % (1 << (t.sh[0] + 1)) == 0) {   // y, z, t exhausted (tiny lattice): give x the rest
        t.sh[0]++;
        vol *= 2;
    }
    t.vol = vol;
    t.ntiles = g.Vh / vol;
    for (int k = 0; k < 3; k++) t.nb[k] = make_fastdiv((unsigned)(ext[k] >> t.sh[k]));
    return t;
}

int choose_zband(int sites_per_plane, int nz, size_t bytes_per_site, size_t l2_budget, int mult)
{
    const double plane3 = 3.0 * (double)sites_per_plane * (double)bytes_per_site;
    if (plane3 * nz <= (double)l2_budget) return 0;
    int best = 0;
    for (int zb = mult; zb < nz; zb += mult)
        if (nz % zb == 0 && plane3 * zb <= (double)l2_budget) best = zb;
    if (best == 0 && mult < nz && nz % mult == 0) best = mult;
    return best;
}

Sweep make_sweep(const Geom &g, int zb)
{
    Sweep w;
    memset(&w, 0, sizeof(w));
    const int plane = g.Xh * g.Y;
    if (zb <= 0 || zb >= g.Z || g.Z % zb != 0 || plane % DSLASH_BLOCK != 0) return w;
    w.on = 1;
    w.zb = zb;
    w.d_up = make_fastdiv((unsigned)(plane / DSLASH_BLOCK));
    w.d_zb = make_fastdiv((unsigned)zb);
    w.d_t = make_fastdiv((unsigned)g.T);
    return w;
}

int mrhs_tile_z(const Geom &g) { return 1 << make_tile(g, MSITES, COLA_MRHS_TILE_X).sh[2]; }
int mrhs_site_blocks(const Geom &g) { return make_tile(g, MSITES, COLA_MRHS_TILE_X).ntiles; }

cudaError_t launch_dslash_mrhs(int fmt, MrhsArgs &m, cudaStream_t s)
{
    if (m.nrhs < 1 || m.nrhs > MRHS_MAX) return cudaErrorInvalidValue;
    switch (fmt) {
        case LINK_F64_18: return launch_mrhs_fmt<LINK_F64_18>(m, s);
        case LINK_F32_18: return launch_mrhs_fmt<LINK_F32_18>(m, s);
        case LINK_F32_12: return launch_mrhs_fmt<LINK_F32_12>(m, s);
        case LINK_I16_12: return launch_mrhs_fmt<LINK_I16_12>(m, s);
        case LINK_F32_8: return launch_mrhs_fmt<LINK_F32_8>(m, s);
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_mrhs_reduce(const double *partials, int nsb, int nrhs, const int *list, double *out, int accumulate, const int *skip, cudaStream_t s)
{
    if (nrhs < 1 || nrhs > MRHS_MAX) return cudaErrorInvalidValue;
    MrhsList l;
    for (int k = 0; k < MRHS_MAX; k++) l.v[k] = k < nrhs ? list[k] : 0;
    mrhs_reduce_kernel<<<nrhs, 256, 0, s>>>(partials, nsb, l, skip, out, accumulate);
    return cudaGetLastError();
}

size_t dslash_grid_blocks(size_t Vh) { return (Vh + DSLASH_BLOCK - 1) / DSLASH_BLOCK; }

cudaError_t launch_dslash(int fmt, const DslashArgs &a, cudaStream_t s)
{
    switch (fmt) {
        case LINK_F64_18: return launch_fmt<LINK_F64_18>(a, s);
        case LINK_F32_18: return launch_fmt<LINK_F32_18>(a, s);
        case LINK_F32_12: return launch_fmt<LINK_F32_12>(a, s);
        case LINK_I16_12: return launch_fmt<LINK_I16_12>(a, s);
        case LINK_F32_8: return launch_fmt<LINK_F32_8>(a, s);
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_clover_apply(cola_prec prec, const Geom &g, const void *clov, const void *in, void *out, cudaStream_t s)
{
    const dim3 grid((g.Vh + DSLASH_BLOCK - 1) / DSLASH_BLOCK), block(DSLASH_BLOCK);
    if (prec == COLA_F64) clover_apply_kernel<double><<<grid, block, 0, s>>>(g.Vh, clov, in, out);
    else clover_apply_kernel<float><<<grid, block, 0, s>>>(g.Vh, clov, in, out);
    return cudaGetLastError();
}

}  // namespace cola
