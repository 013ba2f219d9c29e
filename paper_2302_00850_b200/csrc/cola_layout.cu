// cola_layout.cu -- layout kernels: canonical arrays <-> parity-split SoA of 16-byte
// chunks, fp64 -> fp32 copies, 18 -> 12-real link compression, unitarity diagnostic.
#include "cola_device.cuh"

namespace cola {

namespace {

constexpr int LB = 128;

__device__ __forceinline__ void lex_to_cb(const Geom &g, long lex, int &parity, int &cb)
{
    const int x = (int)(lex % g.X);
    long r = lex / g.X;
    const int y = (int)(r % g.Y);
    r /= g.Y;
    const int z = (int)(r % g.Z);
    const int t = (int)(r / g.Z);
    parity = (x + y + z + t) & 1;
    cb = (x >> 1) + g.Xh * (y + g.Y * (z + g.Z * t));
}

// one thread per (lex site, mu) of the staged canonical chunk
__global__ void __launch_bounds__(LB) gauge_reorder_kernel(Geom g, const double *canon, long site_lo, long n_sites, char *gauge64,
                                                           char *gauge32, int fmt32, char *gauge16, char *gauge8, unsigned long long *max_dev_bits,
                                                           unsigned long long *min_u00_bits)
{
    const long tid = (long)blockIdx.x * LB + threadIdx.x;
    double dev = 0.0, u00 = 2.0;
    if (tid < 4 * n_sites) {
        const long ls = tid >> 2;
        const int mu = (int)(tid & 3);
        const double *src = canon + (ls * 4 + mu) * 18;
        double u[18];
#pragma unroll
        for (int k = 0; k < 18; k++) u[k] = src[k];
        int parity, cb;
        lex_to_cb(g, site_lo + ls, parity, cb);
        const size_t Vh = g.Vh;
        store_reals<double, 18>(gauge64 + (size_t)(parity * 4 + mu) * 144 * Vh, Vh, cb, u);
        char *b32 = gauge32 + (size_t)(parity * 4 + mu) * link_bytes(fmt32) * Vh;
        if (fmt32 == LINK_F32_12) {
            float f[12];
#pragma unroll
            for (int k = 0; k < 12; k++) f[k] = (float)u[k];
            store_reals<float, 12>(b32, Vh, cb, f);
        } else {
            float f[16];
#pragma unroll
            for (int k = 0; k < 16; k++) f[k] = (float)u[k];
            store_reals<float, 16>(b32, Vh, cb, f);
            reinterpret_cast<float2 *>(b32 + 64 * Vh)[cb] = make_float2((float)u[16], (float)u[17]);
        }
        if (gauge16) {   // rows 1, 2 as 16-bit fixed point: round(u * 32767), |u| <= 1 for a unitary matrix (clamped otherwise)
            char *b16 = gauge16 + (size_t)(parity * 4 + mu) * link_bytes(LINK_I16_12) * Vh;
            unsigned w[6];
#pragma unroll
            for (int k = 0; k < 6; k++) {
                const int lo = __double2int_rn(fmin(fmax(u[2 * k], -1.0), 1.0) * 32767.0);
                const int hi = __double2int_rn(fmin(fmax(u[2 * k + 1], -1.0), 1.0) * 32767.0);
                w[k] = ((unsigned)lo & 0xffffu) | ((unsigned)hi << 16);
            }
            reinterpret_cast<uint4 *>(b16)[cb] = make_uint4(w[0], w[1], w[2], w[3]);
            reinterpret_cast<uint2 *>(b16 + 16 * Vh)[cb] = make_uint2(w[4], w[5]);
        }
        u00 = u[0] * u[0] + u[1] * u[1];
        if (gauge8) {   // LINK_F32_8 (cola_internal.h): [a2, a3 | b1, arg(a1)/pi, arg(c1)/pi] with the two flags in the angles' mantissa LSBs
            const double N = u[2] * u[2] + u[3] * u[3] + u[4] * u[4] + u[5] * u[5];
            const bool blockdiag = N < 1e-16;    // |U01|, |U02| < 1e-8: below fp32 resolution of an O(1) entry
            const bool swapped = !blockdiag && (u[6] * u[6] + u[7] * u[7] > u[12] * u[12] + u[13] * u[13]);   // |U10| > |U20|: store (U20, -U10)
            float f[8];
            const double inv_pi = 0.31830988618379067154;
            if (blockdiag) {
                f[0] = (float)u[8]; f[1] = (float)u[9]; f[2] = (float)u[10]; f[3] = (float)u[11];   // U11, U12
                f[4] = 0.0f; f[5] = 0.0f;
                f[7] = 0.0f;
            } else {
                f[0] = (float)u[2]; f[1] = (float)u[3]; f[2] = (float)u[4]; f[3] = (float)u[5];
                const double b1r = swapped ? u[12] : u[6], b1i = swapped ? u[13] : u[7];
                const double c1r = swapped ? -u[6] : u[12], c1i = swapped ? -u[7] : u[13];
                f[4] = (float)b1r; f[5] = (float)b1i;
                f[7] = (float)(atan2(c1i, c1r) * inv_pi);
            }
            f[6] = (float)(atan2(u[1], u[0]) * inv_pi);
            f[6] = __uint_as_float((__float_as_uint(f[6]) & ~1u) | (blockdiag ? 1u : 0u));
            f[7] = __uint_as_float((__float_as_uint(f[7]) & ~1u) | (swapped ? 1u : 0u));
            store_reals<float, 8>(gauge8 + (size_t)(parity * 4 + mu) * link_bytes(LINK_F32_8) * Vh, Vh, cb, f);
        }
        // max |U U^+ - 1| (entry-wise)
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
            for (int b = 0; b < 3; b++) {
                double re = (a == b) ? -1.0 : 0.0, im = 0.0;
#pragma unroll
                for (int c = 0; c < 3; c++) {
                    const double ar = u[2 * (3 * a + c)], ai = u[2 * (3 * a + c) + 1];
                    const double br = u[2 * (3 * b + c)], bi = u[2 * (3 * b + c) + 1];
                    re += ar * br + ai * bi;
                    im += ai * br - ar * bi;
                }
                dev = fmax(dev, sqrt(re * re + im * im));
            }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dev = fmax(dev, __shfl_xor_sync(0xffffffffu, dev, o));
    if ((threadIdx.x & 31) == 0 && dev > 0.0) atomicMax(max_dev_bits, (unsigned long long)__double_as_longlong(dev));
    if (min_u00_bits) {   // min |U00|^2 over all links (non-negative doubles order like their bit patterns): see LINK_F32_8
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) u00 = fmin(u00, __shfl_xor_sync(0xffffffffu, u00, o));
        if ((threadIdx.x & 31) == 0) atomicMin(min_u00_bits, (unsigned long long)__double_as_longlong(u00));
    }
}

template <typename T, bool PACK>
__global__ void __launch_bounds__(LB) spinor_layout_kernel(Geom g, const T *canon_in, T *canon_out, const void *int_in, void *int_out)
{
    const long lex = (long)blockIdx.x * LB + threadIdx.x;
    if (lex >= 2L * g.Vh) return;
    int parity, cb;
    lex_to_cb(g, lex, parity, cb);
    typedef typename VT<T>::V V;
    const size_t half_chunks = (size_t)(24 / VT<T>::N) * g.Vh;
    T r[24];
    if (PACK) {
#pragma unroll
        for (int k = 0; k < 24; k++) r[k] = canon_in[lex * 24 + k];
        store_reals<T, 24>(reinterpret_cast<V *>(int_out) + parity * half_chunks, g.Vh, cb, r);
    } else {
        load_reals<T, 24, true>(reinterpret_cast<const V *>(int_in) + parity * half_chunks, g.Vh, cb, r);
#pragma unroll
        for (int k = 0; k < 24; k++) canon_out[lex * 24 + k] = r[k];
    }
}

// internal fp64 [12 chunks of double2][n] <-> internal fp32 [6 chunks of float4][n]; one thread per (float4 chunk, site)
template <bool TO_F32>
__global__ void __launch_bounds__(LB) convert_kernel(const void *src, void *dst, size_t n)
{
    const size_t tid = (size_t)blockIdx.x * LB + threadIdx.x;
    if (tid >= 6 * n) return;
    const size_t k = tid / n, i = tid - k * n;
    if (TO_F32) {
        const double2 *s = reinterpret_cast<const double2 *>(src);
        const double2 a = s[(2 * k) * n + i], b = s[(2 * k + 1) * n + i];
        reinterpret_cast<float4 *>(dst)[k * n + i] = make_float4((float)a.x, (float)a.y, (float)b.x, (float)b.y);
    } else {
        const float4 v = reinterpret_cast<const float4 *>(src)[k * n + i];
        double2 *d = reinterpret_cast<double2 *>(dst);
        d[(2 * k) * n + i] = make_double2(v.x, v.y);
        d[(2 * k + 1) * n + i] = make_double2(v.z, v.w);
    }
}

}  // namespace

cudaError_t launch_gauge_reorder(const Geom &g, const double *canon_dev, long site_lo, long n_sites, void *gauge64, void *gauge32,
                                 int fmt32, void *gauge16, void *gauge8, unsigned long long *max_dev_bits, unsigned long long *min_u00_bits, cudaStream_t s)
{
    const long n = 4 * n_sites;
    gauge_reorder_kernel<<<(unsigned)((n + LB - 1) / LB), LB, 0, s>>>(g, canon_dev, site_lo, n_sites, (char *)gauge64, (char *)gauge32,
                                                                     fmt32, (char *)gauge16, (char *)gauge8, max_dev_bits, min_u00_bits);
    return cudaGetLastError();
}

cudaError_t launch_spinor_pack(cola_prec prec, const Geom &g, const void *canon, void *internal, cudaStream_t s)
{
    const long n = 2L * g.Vh;
    const unsigned grid = (unsigned)((n + LB - 1) / LB);
    if (prec == COLA_F64) spinor_layout_kernel<double, true><<<grid, LB, 0, s>>>(g, (const double *)canon, nullptr, nullptr, internal);
    else spinor_layout_kernel<float, true><<<grid, LB, 0, s>>>(g, (const float *)canon, nullptr, nullptr, internal);
    return cudaGetLastError();
}

cudaError_t launch_spinor_unpack(cola_prec prec, const Geom &g, const void *internal, void *canon, cudaStream_t s)
{
    const long n = 2L * g.Vh;
    const unsigned grid = (unsigned)((n + LB - 1) / LB);
    if (prec == COLA_F64) spinor_layout_kernel<double, false><<<grid, LB, 0, s>>>(g, nullptr, (double *)canon, internal, nullptr);
    else spinor_layout_kernel<float, false><<<grid, LB, 0, s>>>(g, nullptr, (float *)canon, internal, nullptr);
    return cudaGetLastError();
}

cudaError_t launch_spinor_convert(cola_prec dst_prec, const void *src, void *dst, size_t n_sites, cudaStream_t s)
{
    const size_t n = 6 * n_sites;
    const unsigned grid = (unsigned)((n + LB - 1) / LB);
    if (dst_prec == COLA_F32) convert_kernel<true><<<grid, LB, 0, s>>>(src, dst, n_sites);
    else convert_kernel<false><<<grid, LB, 0, s>>>(src, dst, n_sites);
    return cudaGetLastError();
}

}  // namespace cola
