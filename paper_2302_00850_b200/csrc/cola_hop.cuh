// cola_hop.cuh -- the arithmetic of one hop of the parity dslash, shared by the kernel families in cola_dslash.cu
// (direct global loads) and cola_dslash_tile.cu (neighbour spinors staged in shared memory): spin projection,
// SU(3) x half spinor (H4), reconstruction + accumulation (H5).  Both families call these in the same order, so their
// results are bit-identical (tested).
//
// Chiral basis: gamma_mu = [[0, A_mu], [A_mu^+, 0]], A_k = -i sigma_k, A_t = 1:
//   (1 + s gamma_mu) psi = [ h ; s A_mu^+ h ],   h = psi_upper + s A_mu psi_lower,   s = +-1.
#pragma once
#include "cola_device.cuh"

namespace cola {

// h (2 spins x 3 colours, complex) = upper + s * A_mu * lower of the 24-real spinor p
template <int MU, typename T>
__device__ __forceinline__ void project(const T (&p)[24], T s, T (&h)[12])
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int u0 = 2 * c, u1 = 6 + 2 * c, l0 = 12 + 2 * c, l1 = 18 + 2 * c;   // spin 0,1,2,3 colour c (re)
        if (MU == 0) {          // A = [[0,-i],[-i,0]]
            h[2 * c] = p[u0] + s * p[l1 + 1];
            h[2 * c + 1] = p[u0 + 1] - s * p[l1];
            h[6 + 2 * c] = p[u1] + s * p[l0 + 1];
            h[6 + 2 * c + 1] = p[u1 + 1] - s * p[l0];
        } else if (MU == 1) {   // A = [[0,-1],[1,0]]
            h[2 * c] = p[u0] - s * p[l1];
            h[2 * c + 1] = p[u0 + 1] - s * p[l1 + 1];
            h[6 + 2 * c] = p[u1] + s * p[l0];
            h[6 + 2 * c + 1] = p[u1 + 1] + s * p[l0 + 1];
        } else if (MU == 2) {   // A = [[-i,0],[0,i]]
            h[2 * c] = p[u0] + s * p[l0 + 1];
            h[2 * c + 1] = p[u0 + 1] - s * p[l0];
            h[6 + 2 * c] = p[u1] - s * p[l1 + 1];
            h[6 + 2 * c + 1] = p[u1 + 1] + s * p[l1];
        } else {                // A = 1
            h[2 * c] = p[u0] + s * p[l0];
            h[2 * c + 1] = p[u0 + 1] + s * p[l0 + 1];
            h[6 + 2 * c] = p[u1] + s * p[l1];
            h[6 + 2 * c + 1] = p[u1 + 1] + s * p[l1 + 1];
        }
    }
}

// acc += eta * [ g ; s A_mu^+ g ]
template <int MU, typename T>
__device__ __forceinline__ void reconstruct_accumulate(const T (&g)[12], T eta, T s, T (&acc)[24])
{
    const T se = s * eta;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int u0 = 2 * c, u1 = 6 + 2 * c, l0 = 12 + 2 * c, l1 = 18 + 2 * c;
        const T g0r = g[2 * c], g0i = g[2 * c + 1], g1r = g[6 + 2 * c], g1i = g[6 + 2 * c + 1];
        acc[u0] += eta * g0r;
        acc[u0 + 1] += eta * g0i;
        acc[u1] += eta * g1r;
        acc[u1 + 1] += eta * g1i;
        if (MU == 0) {          // A^+ = [[0,i],[i,0]]: lower0 = i g1, lower1 = i g0
            acc[l0] -= se * g1i;
            acc[l0 + 1] += se * g1r;
            acc[l1] -= se * g0i;
            acc[l1 + 1] += se * g0r;
        } else if (MU == 1) {   // A^+ = [[0,1],[-1,0]]: lower0 = g1, lower1 = -g0
            acc[l0] += se * g1r;
            acc[l0 + 1] += se * g1i;
            acc[l1] -= se * g0r;
            acc[l1 + 1] -= se * g0i;
        } else if (MU == 2) {   // A^+ = [[i,0],[0,-i]]: lower0 = i g0, lower1 = -i g1
            acc[l0] -= se * g0i;
            acc[l0 + 1] += se * g0r;
            acc[l1] += se * g1i;
            acc[l1 + 1] -= se * g1r;
        } else {                // A^+ = 1
            acc[l0] += se * g0r;
            acc[l0 + 1] += se * g0i;
            acc[l1] += se * g1r;
            acc[l1 + 1] += se * g1i;
        }
    }
}

// g = U h (DAG = false) or U^+ h (DAG = true) on both spin components of the half spinor
template <bool DAG, typename T>
__device__ __forceinline__ void su3_mul(const T (&u)[18], const T (&h)[12], T (&g)[12])
{
#pragma unroll
    for (int sp = 0; sp < 2; sp++) {
#pragma unroll
        for (int a = 0; a < 3; a++) {
            T re = 0, im = 0;
#pragma unroll
            for (int b = 0; b < 3; b++) {
                const T ur = DAG ? u[2 * (3 * b + a)] : u[2 * (3 * a + b)];
                const T ui = DAG ? -u[2 * (3 * b + a) + 1] : u[2 * (3 * a + b) + 1];
                const T hr = h[6 * sp + 2 * b], hi = h[6 * sp + 2 * b + 1];
                if (b == 0) {
                    re = fma_(-ui, hi, ur * hr);
                    im = fma_(ui, hr, ur * hi);
                } else {
                    re = fma_(-ui, hi, fma_(ur, hr, re));
                    im = fma_(ui, hr, fma_(ur, hi, im));
                }
            }
            g[6 * sp + 2 * a] = re;
            g[6 * sp + 2 * a + 1] = im;
        }
    }
}

// The epilogues of the fused kernel family on the accumulated hopping term `acc` of output site i:
//   XPAY 1: acc = y + coef acc;  XPAY 2: acc = A y + coef acc;  XPAY 3: the same with A in its 48-real form;
//   POST 1: acc = Cpost acc;  store;  returns |acc|^2 if want_norm.
// STREAM: clover read once per launch (no L1 allocation); !STREAM: shared by the right-hand sides of a block.
// dot (nullable, XPAY != 0 only): dot[0..1] = this site's part of sum conj(out) * y, e.g. BiCGStab's <t, s> for t = S s, whose
// kernel 2 holds s (= y) and t (= out) in registers anyway.
// DOT is a compile-time switch: the kernels without it are the ones of the CGNR iteration and stay as they were.
template <int FMT, int XPAY, int POST, bool STREAM, bool DOT = false>
__device__ __forceinline__ double dslash_epilogue(const DslashArgs &a, const int i, typename LinkT<FMT>::T (&acc)[24], const void *yin, void *out,
                                                  const bool want_norm, double *dot = nullptr)
{
    typedef typename LinkT<FMT>::T T;
    const size_t Vh = a.g.Vh;
    double nrm = 0.0;
    T yv[24];
    if (XPAY != 0) {
        load_reals<T, 24, true>(yin, Vh, i, yv);
        const T cf = (T)a.coef;
        if (XPAY == 2 || XPAY == 3) {
            T cy[24];
            if constexpr (XPAY == 3) clover_apply_g48<T, STREAM>(a.clov_y, Vh, i, yv, cy);
            else clover_apply<T, STREAM, FMT == LINK_I16_12>(a.clov_y, Vh, i, yv, cy);
#pragma unroll
            for (int k = 0; k < 24; k++) acc[k] = cy[k] + cf * acc[k];
        } else {
#pragma unroll
            for (int k = 0; k < 24; k++) acc[k] = yv[k] + cf * acc[k];
        }
    }
    if (POST != 0) {
        T w[24];
        clover_apply<T, STREAM, FMT == LINK_I16_12>(a.clov_post, Vh, i, acc, w);
#pragma unroll
        for (int k = 0; k < 24; k++) acc[k] = w[k];
    }
    store_reals<T, 24>(out, Vh, i, acc);
    if (want_norm) {
        T s2 = 0;
#pragma unroll
        for (int k = 0; k < 24; k++) s2 += acc[k] * acc[k];
        nrm = (double)s2;
        if constexpr (XPAY != 0 && DOT) {
            T dr = 0, di = 0;
#pragma unroll
            for (int k = 0; k < 12; k++) {
                dr += acc[2 * k] * yv[2 * k] + acc[2 * k + 1] * yv[2 * k + 1];
                di += acc[2 * k] * yv[2 * k + 1] - acc[2 * k + 1] * yv[2 * k];
            }
            dot[0] = (double)dr;
            dot[1] = (double)di;
        }
    }
    return nrm;
}

}  // namespace cola
