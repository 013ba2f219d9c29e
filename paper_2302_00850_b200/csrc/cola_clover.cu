// cola_clover.cu -- setup kernels for the clover term (8(c) O4), fp64.
//
// H1: per site, F_{mu nu} from the four-leaf clover average of plaquettes, then the two 6x6
//     Hermitian chiral blocks of A = 1 - kappa*csw*sum_{mu<nu} sigma_{mu nu} (x) F_{mu nu}.
//     In the chiral basis sigma_{mu nu} is block diagonal, so with
//         upper: B1 = F_xt - F_yz, B2 = F_xz + F_yt, B3 = F_zt - F_xy
//         lower: B1 = -F_xt - F_yz, B2 = F_xz - F_yt, B3 = -F_zt - F_xy
//     each block is 1 - k [[B3, B1 - i B2], [B1 + i B2, -B3]]  (spin slow, colour fast).
// H2: per site and block, 6x6 Hermitian positive-definite inverse (Gauss-Jordan, fp64).
// Packed storage: per block 6 real diagonal entries, then the 15 strictly-lower complex entries
// row by row; 72 reals per site as [chunk][Vh] like every other field.
#include "cola_device.cuh"

namespace cola {

namespace {

constexpr int CB = 64;

struct M3 {
    double r[9], i[9];
};

__device__ __forceinline__ void m3_mul(M3 &c, const M3 &a, const M3 &b)   // c = a b
{
    M3 t;
#pragma unroll
    for (int x = 0; x < 3; x++)
#pragma unroll
        for (int y = 0; y < 3; y++) {
            double re = 0, im = 0;
#pragma unroll
            for (int k = 0; k < 3; k++) {
                re += a.r[3 * x + k] * b.r[3 * k + y] - a.i[3 * x + k] * b.i[3 * k + y];
                im += a.r[3 * x + k] * b.i[3 * k + y] + a.i[3 * x + k] * b.r[3 * k + y];
            }
            t.r[3 * x + y] = re;
            t.i[3 * x + y] = im;
        }
    c = t;
}

__device__ __forceinline__ M3 m3_dag(const M3 &a)
{
    M3 t;
#pragma unroll
    for (int x = 0; x < 3; x++)
#pragma unroll
        for (int y = 0; y < 3; y++) {
            t.r[3 * x + y] = a.r[3 * y + x];
            t.i[3 * x + y] = -a.i[3 * y + x];
        }
    return t;
}

// link U_mu at lattice coordinates c (wrapped by the caller) from the internal fp64 gauge field
__device__ __forceinline__ M3 link_at(const Geom &g, const char *gauge64, const int (&c)[4], int mu)
{
    const int parity = (c[0] + c[1] + c[2] + c[3]) & 1;
    const int cb = (c[0] >> 1) + g.Xh * (c[1] + g.Y * (c[2] + g.Z * c[3]));
    double u[18];
    load_reals<double, 18, false>(gauge64 + (size_t)(parity * 4 + mu) * 144 * g.Vh, g.Vh, cb, u);
    M3 m;
#pragma unroll
    for (int k = 0; k < 9; k++) {
        m.r[k] = u[2 * k];
        m.i[k] = u[2 * k + 1];
    }
    return m;
}

__device__ __forceinline__ void shifted(const Geom &g, const int (&c)[4], int mu, int d0, int nu, int d1, int (&o)[4])
{
    const int L[4] = {g.X, g.Y, g.Z, g.T};
#pragma unroll
    for (int k = 0; k < 4; k++) o[k] = c[k];
    o[mu] = (o[mu] + d0 + L[mu]) % L[mu];
    o[nu] = (o[nu] + d1 + L[nu]) % L[nu];
}

// F_{mu nu}(x), Hermitian (traceless if trace_sub)
__device__ void field_strength(const Geom &g, const char *gauge64, const int (&c)[4], int mu, int nu, int trace_sub, M3 &F)
{
    int xpm[4], xpn[4], xmm[4], xmn[4], xmmpn[4], xmmmn[4], xpmmn[4];
    shifted(g, c, mu, +1, nu, 0, xpm);
    shifted(g, c, mu, 0, nu, +1, xpn);
    shifted(g, c, mu, -1, nu, 0, xmm);
    shifted(g, c, mu, 0, nu, -1, xmn);
    shifted(g, c, mu, -1, nu, +1, xmmpn);
    shifted(g, c, mu, -1, nu, -1, xmmmn);
    shifted(g, c, mu, +1, nu, -1, xpmmn);
    M3 Q, leaf;
    // leaf 1: U_mu(x) U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+
    m3_mul(leaf, link_at(g, gauge64, c, mu), link_at(g, gauge64, xpm, nu));
    m3_mul(leaf, leaf, m3_dag(link_at(g, gauge64, xpn, mu)));
    m3_mul(leaf, leaf, m3_dag(link_at(g, gauge64, c, nu)));
    Q = leaf;
    // leaf 2: U_nu(x) U_mu(x-mu+nu)^+ U_nu(x-mu)^+ U_mu(x-mu)
    m3_mul(leaf, link_at(g, gauge64, c, nu), m3_dag(link_at(g, gauge64, xmmpn, mu)));
    m3_mul(leaf, leaf, m3_dag(link_at(g, gauge64, xmm, nu)));
    m3_mul(leaf, leaf, link_at(g, gauge64, xmm, mu));
#pragma unroll
    for (int k = 0; k < 9; k++) { Q.r[k] += leaf.r[k]; Q.i[k] += leaf.i[k]; }
    // leaf 3: U_mu(x-mu)^+ U_nu(x-mu-nu)^+ U_mu(x-mu-nu) U_nu(x-nu)
    m3_mul(leaf, m3_dag(link_at(g, gauge64, xmm, mu)), m3_dag(link_at(g, gauge64, xmmmn, nu)));
    m3_mul(leaf, leaf, link_at(g, gauge64, xmmmn, mu));
    m3_mul(leaf, leaf, link_at(g, gauge64, xmn, nu));
#pragma unroll
    for (int k = 0; k < 9; k++) { Q.r[k] += leaf.r[k]; Q.i[k] += leaf.i[k]; }
    // leaf 4: U_nu(x-nu)^+ U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^+
    m3_mul(leaf, m3_dag(link_at(g, gauge64, xmn, nu)), link_at(g, gauge64, xmn, mu));
    m3_mul(leaf, leaf, link_at(g, gauge64, xpmmn, nu));
    m3_mul(leaf, leaf, m3_dag(link_at(g, gauge64, c, mu)));
#pragma unroll
    for (int k = 0; k < 9; k++) { Q.r[k] += leaf.r[k]; Q.i[k] += leaf.i[k]; }
    // G = (Q - Q^+)/8 (anti-Hermitian); F = -i (G - tr G/3):  F.re = G.im, F.im = -G.re
    double tr_im = 0.0;
#pragma unroll
    for (int a = 0; a < 3; a++) tr_im += 2.0 * Q.i[4 * a] / 8.0;   // tr G is purely imaginary
    const double sub = trace_sub ? tr_im / 3.0 : 0.0;
#pragma unroll
    for (int a = 0; a < 3; a++)
#pragma unroll
        for (int b = 0; b < 3; b++) {
            const double g_re = (Q.r[3 * a + b] - Q.r[3 * b + a]) / 8.0;
            const double g_im = (Q.i[3 * a + b] + Q.i[3 * b + a]) / 8.0 - (a == b ? sub : 0.0);
            F.r[3 * a + b] = g_im;
            F.i[3 * a + b] = -g_re;
        }
}

// pack a full Hermitian 6x6 (re, im arrays, row-major) into 36 reals
__device__ __forceinline__ void pack_block(const double (&br)[36], const double (&bi)[36], double (&p)[36])
{
#pragma unroll
    for (int i = 0; i < 6; i++) p[i] = br[7 * i];
#pragma unroll
    for (int i = 1; i < 6; i++)
#pragma unroll
        for (int j = 0; j < i; j++) {
            const int k = 6 + 2 * (i * (i - 1) / 2 + j);
            p[k] = br[6 * i + j];
            p[k + 1] = bi[6 * i + j];
        }
}

__device__ __forceinline__ unsigned pack_h16(double a, double b)
{
    const __half2 h = __floats2half2_rn((float)a, (float)b);
    return *reinterpret_cast<const unsigned *>(&h);
}

__device__ __forceinline__ void store_block(char *c64, char *c32, char *c16, size_t Vh, int blk, size_t i, const double (&p)[36])
{
    store_reals<double, 36>(reinterpret_cast<double2 *>(c64) + (size_t)blk * 18 * Vh, Vh, i, p);
    if (c16) {   // fp16 copy: per block 4 chunks of 8 halfs + 1 chunk of 4 halfs (clover_apply<.., H16> in cola_device.cuh)
        char *base = c16 + (size_t)blk * 72 * Vh;
#pragma unroll
        for (int k = 0; k < 4; k++)
            reinterpret_cast<uint4 *>(base + (size_t)k * 16 * Vh)[i] =
                make_uint4(pack_h16(p[8 * k], p[8 * k + 1]), pack_h16(p[8 * k + 2], p[8 * k + 3]), pack_h16(p[8 * k + 4], p[8 * k + 5]), pack_h16(p[8 * k + 6], p[8 * k + 7]));
        reinterpret_cast<uint2 *>(base + (size_t)64 * Vh)[i] = make_uint2(pack_h16(p[32], p[33]), pack_h16(p[34], p[35]));
    }
    if (c32) {
        float f[36];
#pragma unroll
        for (int k = 0; k < 36; k++) f[k] = (float)p[k];
        store_reals<float, 36>(reinterpret_cast<float4 *>(c32) + (size_t)blk * 9 * Vh, Vh, i, f);
    }
}

// one thread per site: tid < 2*Vh, parity = tid / Vh
__global__ void __launch_bounds__(CB) clover_build_kernel(Geom g, const char *gauge64, double k, int trace_sub, char *A64, char *A32, int a32_parities, char *A16,
                                                          char *G32)
{
    const long tid = (long)blockIdx.x * CB + threadIdx.x;
    if (tid >= 2L * g.Vh) return;
    const int parity = (int)(tid / g.Vh);
    const int i = (int)(tid - (long)parity * g.Vh);
    int c[4];
    {
        const int xh = i % g.Xh;
        int r = i / g.Xh;
        c[1] = r % g.Y;
        r /= g.Y;
        c[2] = r % g.Z;
        c[3] = r / g.Z;
        c[0] = 2 * xh + ((c[1] + c[2] + c[3] + parity) & 1);
    }
    M3 Fxy, Fxz, Fxt, Fyz, Fyt, Fzt;
    field_strength(g, gauge64, c, 0, 1, trace_sub, Fxy);
    field_strength(g, gauge64, c, 0, 2, trace_sub, Fxz);
    field_strength(g, gauge64, c, 0, 3, trace_sub, Fxt);
    field_strength(g, gauge64, c, 1, 2, trace_sub, Fyz);
    field_strength(g, gauge64, c, 1, 3, trace_sub, Fyt);
    field_strength(g, gauge64, c, 2, 3, trace_sub, Fzt);
    const size_t Vh = g.Vh;
    char *a64 = A64 + (size_t)parity * 72 * 8 * Vh;
    char *a32 = (A32 && parity < a32_parities) ? A32 + (size_t)parity * 72 * 4 * Vh : nullptr;   // fp32 A on the odd parity is optional
    char *a16 = (A16 && parity < a32_parities) ? A16 + (size_t)parity * CLOVER_H16_BYTES * Vh : nullptr;
    char *g32 = (G32 && parity < a32_parities) ? G32 + (size_t)parity * CLOVER_G48_REALS * 4 * Vh : nullptr;
#pragma unroll
    for (int blk = 0; blk < 2; blk++) {
        const double sg = blk == 0 ? 1.0 : -1.0;
        if (g32) {   // 48-real form: G_j = -k B_j as [d0, d1, l10, l20, l21], order G3, G1, G2 (load_clover_g48 in cola_device.cuh)
            float f[24];
            const int e_of[5] = {0, 4, 3, 6, 7};   // (0,0) (1,1) | (1,0) (2,0) (2,1) in row-major 3x3
#pragma unroll
            for (int q = 0; q < 5; q++) {
                const int e = e_of[q];
                const double B1r = sg * Fxt.r[e] - Fyz.r[e], B1i = sg * Fxt.i[e] - Fyz.i[e];
                const double B2r = Fxz.r[e] + sg * Fyt.r[e], B2i = Fxz.i[e] + sg * Fyt.i[e];
                const double B3r = sg * Fzt.r[e] - Fxy.r[e], B3i = sg * Fzt.i[e] - Fxy.i[e];
                if (q < 2) {
                    f[q] = (float)(-k * B3r); f[8 + q] = (float)(-k * B1r); f[16 + q] = (float)(-k * B2r);
                } else {
                    const int o = 2 + 2 * (q - 2);
                    f[o] = (float)(-k * B3r); f[o + 1] = (float)(-k * B3i);
                    f[8 + o] = (float)(-k * B1r); f[8 + o + 1] = (float)(-k * B1i);
                    f[16 + o] = (float)(-k * B2r); f[16 + o + 1] = (float)(-k * B2i);
                }
            }
            store_reals<float, 24>(reinterpret_cast<float4 *>(g32) + (size_t)blk * 6 * Vh, Vh, i, f);
        }
        double br[36], bi[36];
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
            for (int b = 0; b < 3; b++) {
                const int e = 3 * a + b;
                const double B1r = sg * Fxt.r[e] - Fyz.r[e], B1i = sg * Fxt.i[e] - Fyz.i[e];
                const double B2r = Fxz.r[e] + sg * Fyt.r[e], B2i = Fxz.i[e] + sg * Fyt.i[e];
                const double B3r = sg * Fzt.r[e] - Fxy.r[e], B3i = sg * Fzt.i[e] - Fxy.i[e];
                const double d = (a == b) ? 1.0 : 0.0;
                // [[B3, B1 - iB2], [B1 + iB2, -B3]]
                br[6 * a + b] = d - k * B3r;
                bi[6 * a + b] = -k * B3i;
                br[6 * (3 + a) + 3 + b] = d + k * B3r;
                bi[6 * (3 + a) + 3 + b] = k * B3i;
                br[6 * a + 3 + b] = -k * (B1r + B2i);
                bi[6 * a + 3 + b] = -k * (B1i - B2r);
                br[6 * (3 + a) + b] = -k * (B1r - B2i);
                bi[6 * (3 + a) + b] = -k * (B1i + B2r);
            }
        double p[36];
        pack_block(br, bi, p);
        store_block(a64, a32, a16, Vh, blk, i, p);
    }
}

// one thread per (site, block) of one parity: tid < 2*Vh, blk = tid / Vh
// order-preserving map of a double onto unsigned 64-bit keys (atomicMin on the key = min of the doubles, any sign)
__device__ __forceinline__ unsigned long long order_key(double v)
{
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}

__global__ void __launch_bounds__(CB) clover_invert_kernel(Geom g, const char *A64, char *I64, char *I32, char *I16, unsigned long long *min_pivot_key)
{
    const long tid = (long)blockIdx.x * CB + threadIdx.x;
    unsigned long long key = ~0ull;    // threads past the end take part in the warp minimum with the neutral key
    if (tid < 2L * g.Vh) {
    const int blk = (int)(tid / g.Vh);
    const int i = (int)(tid - (long)blk * g.Vh);
    const size_t Vh = g.Vh;
    double p[36];
    load_reals<double, 36, true>(reinterpret_cast<const double2 *>(A64) + (size_t)blk * 18 * Vh, Vh, i, p);
    double ar[36], ai[36];
    for (int r = 0; r < 6; r++) {
        ar[7 * r] = p[r];
        ai[7 * r] = 0.0;
        for (int c = 0; c < r; c++) {
            const int k = 6 + 2 * (r * (r - 1) / 2 + c);
            ar[6 * r + c] = p[k];
            ai[6 * r + c] = p[k + 1];
            ar[6 * c + r] = p[k];
            ai[6 * c + r] = -p[k + 1];
        }
    }
    // in-place Gauss-Jordan inverse without pivoting (Hermitian positive definite: pivots are real > 0 up to rounding).
    // The smallest pivot met is reported; a pivot <= 0 means the block is not positive definite.
    double pmin = 1e300;
    for (int c = 0; c < 6; c++) {
        const double pr = ar[7 * c], pi = ai[7 * c];
        pmin = (pr < pmin || !(pr == pr)) ? pr : pmin;
        const double den = 1.0 / (pr * pr + pi * pi);
        const double ir = pr * den, ii = -pi * den;   // 1/pivot
        ar[7 * c] = 1.0;
        ai[7 * c] = 0.0;
        for (int j = 0; j < 6; j++) {
            const double xr = ar[6 * c + j], xi = ai[6 * c + j];
            ar[6 * c + j] = xr * ir - xi * ii;
            ai[6 * c + j] = xr * ii + xi * ir;
        }
        for (int r = 0; r < 6; r++) {
            if (r == c) continue;
            const double fr = ar[6 * r + c], fi = ai[6 * r + c];
            ar[6 * r + c] = 0.0;
            ai[6 * r + c] = 0.0;
            for (int j = 0; j < 6; j++) {
                ar[6 * r + j] -= fr * ar[6 * c + j] - fi * ai[6 * c + j];
                ai[6 * r + j] -= fr * ai[6 * c + j] + fi * ar[6 * c + j];
            }
        }
    }
    double q[36];
    pack_block(ar, ai, q);
    store_block(I64, I32, I16, Vh, blk, i, q);
    key = (pmin == pmin) ? order_key(pmin) : 0ull;   // NaN pivots map to a key below every number's (reported as not positive definite)
    }
    if (min_pivot_key) {
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long other = __shfl_xor_sync(0xffffffffu, key, o);
            key = other < key ? other : key;
        }
        if ((threadIdx.x & 31) == 0) atomicMin(min_pivot_key, key);
    }
}

// expand packed blocks to canonical 12x12 complex per lex site; parity_mask bit p set => parity p is
// present at clov64 + (index among present parities)*72*8*Vh, absent parities give zero blocks
__global__ void __launch_bounds__(CB) clover_unpack_kernel(Geom g, const char *clov64, int parity_mask, double *canon)
{
    const long lex = (long)blockIdx.x * CB + threadIdx.x;
    if (lex >= 2L * g.Vh) return;
    const int x = (int)(lex % g.X);
    long r = lex / g.X;
    const int y = (int)(r % g.Y);
    r /= g.Y;
    const int z = (int)(r % g.Z);
    const int t = (int)(r / g.Z);
    const int parity = (x + y + z + t) & 1;
    const int cb = (x >> 1) + g.Xh * (y + g.Y * (z + g.Z * t));
    double *out = canon + lex * 288;
    for (int k = 0; k < 288; k++) out[k] = 0.0;
    if (!((parity_mask >> parity) & 1)) return;
    const int slot = (parity == 1 && (parity_mask & 1)) ? 1 : 0;
    const size_t Vh = g.Vh;
    const char *base = clov64 + (size_t)slot * 72 * 8 * Vh;
    for (int blk = 0; blk < 2; blk++) {
        double p[36];
        load_reals<double, 36, true>(reinterpret_cast<const double2 *>(base) + (size_t)blk * 18 * Vh, Vh, cb, p);
        for (int a = 0; a < 6; a++) {
            const int row = 6 * blk + a;
            out[2 * (12 * row + row)] = p[a];
            for (int b = 0; b < a; b++) {
                const int k = 6 + 2 * (a * (a - 1) / 2 + b);
                const int col = 6 * blk + b;
                out[2 * (12 * row + col)] = p[k];
                out[2 * (12 * row + col) + 1] = p[k + 1];
                out[2 * (12 * col + row)] = p[k];
                out[2 * (12 * col + row) + 1] = -p[k + 1];
            }
        }
    }
}

}  // namespace

cudaError_t launch_clover_build(const Geom &g, const void *gauge64, double kappa_csw, int trace_sub, void *clovA64, void *clovA32, int a32_parities, void *clovA16,
                                void *clovG32, cudaStream_t s)
{
    const long n = 2L * g.Vh;
    clover_build_kernel<<<(unsigned)((n + CB - 1) / CB), CB, 0, s>>>(g, (const char *)gauge64, kappa_csw, trace_sub, (char *)clovA64, (char *)clovA32, a32_parities, (char *)clovA16,
                                                                     (char *)clovG32);
    return cudaGetLastError();
}

cudaError_t launch_clover_invert(const Geom &g, const void *clovA64_odd, void *clovI64, void *clovI32, void *clovI16, unsigned long long *min_pivot_key, cudaStream_t s)
{
    const long n = 2L * g.Vh;
    clover_invert_kernel<<<(unsigned)((n + CB - 1) / CB), CB, 0, s>>>(g, (const char *)clovA64_odd, (char *)clovI64, (char *)clovI32, (char *)clovI16, min_pivot_key);
    return cudaGetLastError();
}

cudaError_t launch_clover_unpack(const Geom &g, const void *clov64, int parity_mask, void *canon, cudaStream_t s)
{
    const long n = 2L * g.Vh;
    clover_unpack_kernel<<<(unsigned)((n + CB - 1) / CB), CB, 0, s>>>(g, (const char *)clov64, parity_mask, (double *)canon);
    return cudaGetLastError();
}

}  // namespace cola
