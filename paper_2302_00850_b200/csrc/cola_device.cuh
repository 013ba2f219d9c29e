// cola_device.cuh -- device-side building blocks: 16-byte SoA chunk I/O, SU(3) link load with
// in-register third-row reconstruction (BJ:ns), packed 6x6 Hermitian clover mat-vec,
// deterministic warp-shuffle + block + last-block reduction.
#pragma once
#include <cuda_fp16.h>

#include "cola_internal.h"

namespace cola {

// Programmatic dependent launch (sm_90+): a kernel launched with launch_pdl may be scheduled while its predecessor in
// the stream is still draining.  pdl_trigger() at the top of the predecessor says "my blocks have all started", so the
// successor's blocks take the SM slots the predecessor's last wave leaves free; pdl_wait() in the successor blocks
// until the predecessor has completed and its writes are visible.  Every kernel launched through launch_pdl calls
// pdl_wait() before it touches memory.  Without the launch attribute both are no-ops.
#ifndef COLA_PDL
#define COLA_PDL 1
#endif
__device__ __forceinline__ void pdl_trigger()
{
#if COLA_PDL
    asm volatile("griddepcontrol.launch_dependents;");
#endif
}
__device__ __forceinline__ void pdl_wait()
{
#if COLA_PDL
    asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
}
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl_smem(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, Args... args)
{
#if COLA_PDL
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
#else
    kern<<<grid, block, smem, s>>>(args...);
    return cudaGetLastError();
#endif
}
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, cudaStream_t s, Args... args)
{
    return launch_pdl_smem(kern, grid, block, 0, s, args...);
}

// Asynchronous 16-byte copy global -> shared (LDGSTS): the data in flight needs no destination register.  A thread that
// only reads back what it copied itself needs no barrier: cp_async_wait<N>() returns when all but the N most recently
// committed groups of THIS thread have landed.
__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <typename T> struct VT;
template <> struct VT<float> {
    typedef float4 V;
    static constexpr int N = 4;
};
template <> struct VT<double> {
    typedef double2 V;
    static constexpr int N = 2;
};

// ---- 16-byte global loads/stores.  "stream" = read-once data (links, clover): bypass L1 allocation
// so that L1 keeps the neighbour spinors, which are the only data with reuse inside a block.
__device__ __forceinline__ float4 ld_stream(const float4 *p)
{
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ float2 ld_stream(const float2 *p)
{
    float2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0,%1}, [%2];" : "=f"(r.x), "=f"(r.y) : "l"(p));
    return r;
}
__device__ __forceinline__ double2 ld_stream(const double2 *p)
{
    double2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
    return r;
}
__device__ __forceinline__ uint4 ld_stream(const uint4 *p)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ uint2 ld_stream(const uint2 *p)
{
    uint2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "l"(p));
    return r;
}
__device__ __forceinline__ float4 ld_cached(const float4 *p) { return __ldg(p); }
__device__ __forceinline__ double2 ld_cached(const double2 *p) { return __ldg(p); }

// Explicit fused multiply-add chains: without fast-math the compiler may not reassociate `re += a*b - c*d`
// into two dependent FMAs (it emits FMUL + FFMA + FADD), and the fp32 kernels are close to issue-bound.
__device__ __forceinline__ float fma_(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ double fma_(double a, double b, double c) { return __fma_rn(a, b, c); }

__device__ __forceinline__ void unpack(const float4 &v, float *r) { r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w; }
__device__ __forceinline__ void unpack(const double2 &v, double *r) { r[0] = v.x; r[1] = v.y; }
__device__ __forceinline__ float4 pack(const float *r) { return make_float4(r[0], r[1], r[2], r[3]); }
__device__ __forceinline__ double2 pack(const double *r) { return make_double2(r[0], r[1]); }

// NR reals of site i from an SoA field of 16-byte chunks with chunk stride `stride` (in chunks)
template <typename T, int NR, bool STREAM>
__device__ __forceinline__ void load_reals(const void *base, size_t stride, size_t i, T (&r)[NR])
{
    typedef typename VT<T>::V V;
    constexpr int N = VT<T>::N;
    const V *p = reinterpret_cast<const V *>(base) + i;
#pragma unroll
    for (int k = 0; k < NR / N; k++) {
        V v = STREAM ? ld_stream(p + (size_t)k * stride) : ld_cached(p + (size_t)k * stride);
        unpack(v, &r[k * N]);
    }
}

template <typename T, int NR>
__device__ __forceinline__ void store_reals(void *base, size_t stride, size_t i, const T (&r)[NR])
{
    typedef typename VT<T>::V V;
    constexpr int N = VT<T>::N;
    V *p = reinterpret_cast<V *>(base) + i;
#pragma unroll
    for (int k = 0; k < NR / N; k++) p[(size_t)k * stride] = pack(&r[k * N]);
}

// ---- links.  u[18] = row-major (re, im) of the 3x3 matrix.
// third row of an SU(3) matrix from the first two: row3 = conj(row1 x row2)
template <typename T>
__device__ __forceinline__ void reconstruct_row3(T (&u)[18])
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        // U_2c = conj(U_0a U_1b - U_0b U_1a)
        const T ar = u[2 * a], ai = u[2 * a + 1], br = u[2 * b], bi = u[2 * b + 1];                  // row 1
        const T cr = u[6 + 2 * b], ci = u[6 + 2 * b + 1], dr = u[6 + 2 * a], di = u[6 + 2 * a + 1];  // row 2
        // re = ar cr - ai ci - br dr + bi di;  -im = -(ar ci + ai cr - br di - bi dr)
        u[12 + 2 * c] = fma_(bi, di, fma_(-br, dr, fma_(-ai, ci, ar * cr)));
        u[12 + 2 * c + 1] = fma_(bi, dr, fma_(br, di, fma_(-ai, cr, -(ar * ci))));
    }
}

template <int FMT> struct LinkT;
template <> struct LinkT<LINK_F64_18> { typedef double T; };
template <> struct LinkT<LINK_F32_18> { typedef float T; };
template <> struct LinkT<LINK_F32_12> { typedef float T; };
template <> struct LinkT<LINK_I16_12> { typedef float T; };
template <> struct LinkT<LINK_F32_8> { typedef float T; };

// two 16-bit fixed-point reals (x 32767) of one 32-bit word
__device__ __forceinline__ void unpack_i16(unsigned w, float &a, float &b)
{
    constexpr float inv = 1.0f / 32767.0f;
    a = (float)(short)(w & 0xffffu) * inv;
    b = (float)(short)(w >> 16) * inv;
}
__device__ __forceinline__ void unpack_h16(unsigned w, float &a, float &b)
{
    const float2 f = __half22float2(*reinterpret_cast<const __half2 *>(&w));
    a = f.x;
    b = f.y;
}

// A link as it sits in memory (raw) and its expansion to the 18 reals of the 3x3 matrix.  Split in two so that the
// load of the NEXT hop's link can be issued while the current hop is still computing (software pipelining): the raw
// words are all that has to stay live.
template <int FMT> struct RawLink;
template <> struct RawLink<LINK_F64_18> { double r[18]; };
template <> struct RawLink<LINK_F32_18> { float r[18]; };
template <> struct RawLink<LINK_F32_12> { float r[12]; };
template <> struct RawLink<LINK_I16_12> { unsigned w[6]; };
template <> struct RawLink<LINK_F32_8> { float r[8]; };

// ---- 8-real links (LINK_F32_8; layout and flags in cola_internal.h).  With row 1 = (a1, a2, a3), N = |a2|^2 + |a3|^2,
// |a1| = sqrt(1 - N), (b1, c1) the first-column entries of rows 2 and 3, |c1| = sqrt(N - |b1|^2), unitarity and det = 1 give
//   b2 = x a2 + y conj(a3),  b3 = x a3 - y conj(a2),   x  = -conj(a1) b1 / N,  y  = -conj(c1) / N,
//   c2 = x' a2 + y' conj(a3), c3 = x' a3 - y' conj(a2),  x' = -conj(a1) c1 / N,  y' =  conj(b1) / N.
// MUFU approximations (sin/cos, rcp, sqrt) are accurate to ~4e-7 absolute on a link entry: "additional computation
// in order to reduce traffic from global memory".  COLA_R8_EXACT_TRIG = 1 uses sincospif instead.
#ifndef COLA_R8_EXACT_TRIG
#define COLA_R8_EXACT_TRIG 0
#endif
__device__ __forceinline__ float rcp_approx(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float sqrt_approx(float x)
{
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ void sincospi_(float x, float &sn, float &cs)
{
#if COLA_R8_EXACT_TRIG
    sincospif(x, &sn, &cs);
#else
    __sincosf(3.14159265358979323846f * x, &sn, &cs);
#endif
}
__device__ __forceinline__ void reconstruct8(const float (&s)[8], float (&u)[18])
{
    const float a2r = s[0], a2i = s[1], a3r = s[2], a3i = s[3], b1r = s[4], b1i = s[5];
    const bool blockdiag = (__float_as_uint(s[6]) & 1u) != 0u, swapped = (__float_as_uint(s[7]) & 1u) != 0u;
    float s1, c1, s2, c2;
    sincospi_(s[6], s1, c1);
    sincospi_(s[7], s2, c2);
    if (blockdiag) {   // U = [[e, 0, 0], [0, p, q], [0, -conj(q) conj(e), conj(p) conj(e)]], e = exp(i th1), p, q in the a2, a3 slots
        u[0] = c1; u[1] = s1; u[2] = 0; u[3] = 0; u[4] = 0; u[5] = 0;
        u[6] = 0; u[7] = 0; u[8] = a2r; u[9] = a2i; u[10] = a3r; u[11] = a3i;
        u[12] = 0; u[13] = 0;
        u[14] = a3i * s1 - a3r * c1; u[15] = a3r * s1 + a3i * c1;
        u[16] = a2r * c1 - a2i * s1; u[17] = -(a2r * s1 + a2i * c1);
        return;
    }
    const float N = fma_(a2r, a2r, fma_(a2i, a2i, fma_(a3r, a3r, a3i * a3i)));
    const float rN = rcp_approx(N);
    const float m1 = sqrt_approx(fmaxf(1.0f - N, 0.0f));
    const float mc = sqrt_approx(fmaxf(fma_(-b1r, b1r, fma_(-b1i, b1i, N)), 0.0f));
    const float a1r = m1 * c1, a1i = m1 * s1, c1r = mc * c2, c1i = mc * s2;
    const float xr = -rN * fma_(a1r, b1r, a1i * b1i), xi = -rN * fma_(a1r, b1i, -(a1i * b1r));
    const float pr = -rN * fma_(a1r, c1r, a1i * c1i), pi = -rN * fma_(a1r, c1i, -(a1i * c1r));
    const float yr = -rN * c1r, yi = rN * c1i;
    const float qr = rN * b1r, qi = -rN * b1i;
    // z a2 + w conj(a3),  z a3 - w conj(a2)
    const float b2r = fma_(yi, a3i, fma_(yr, a3r, fma_(-xi, a2i, xr * a2r))), b2i = fma_(yi, a3r, fma_(-yr, a3i, fma_(xi, a2r, xr * a2i)));
    const float b3r = fma_(-yi, a2i, fma_(-yr, a2r, fma_(-xi, a3i, xr * a3r))), b3i = fma_(-yi, a2r, fma_(yr, a2i, fma_(xi, a3r, xr * a3i)));
    const float c2r = fma_(qi, a3i, fma_(qr, a3r, fma_(-pi, a2i, pr * a2r))), c2i = fma_(qi, a3r, fma_(-qr, a3i, fma_(pi, a2r, pr * a2i)));
    const float c3r = fma_(-qi, a2i, fma_(-qr, a2r, fma_(-pi, a3i, pr * a3r))), c3i = fma_(-qi, a2r, fma_(qr, a2i, fma_(pi, a3r, pr * a3i)));
    u[0] = a1r; u[1] = a1i; u[2] = a2r; u[3] = a2i; u[4] = a3r; u[5] = a3i;
    const float rb[6] = {b1r, b1i, b2r, b2i, b3r, b3i}, rc[6] = {c1r, c1i, c2r, c2i, c3r, c3i};
#pragma unroll
    for (int k = 0; k < 6; k++) {   // swapped: the stored pair was (U20, -U10): row 2 = -rc, row 3 = rb
        u[6 + k] = swapped ? -rc[k] : rb[k];
        u[12 + k] = swapped ? rb[k] : rc[k];
    }
}

// base = start of the [chunk][Vh] block of one (parity, mu)
// STREAM: read-once data, no L1 allocation (single right-hand side); !STREAM: the same link is read by the
// threads of several right-hand sides of one block, so it is kept in L1.
template <int FMT, bool STREAM = true>
__device__ __forceinline__ void load_raw_link(const char *base, size_t Vh, size_t i, RawLink<FMT> &raw)
{
    if constexpr (FMT == LINK_F64_18) {
        load_reals<double, 18, STREAM>(base, Vh, i, raw.r);
    } else if constexpr (FMT == LINK_I16_12) {
        const uint4 *pa = reinterpret_cast<const uint4 *>(base) + i;
        const uint2 *pb = reinterpret_cast<const uint2 *>(base + 16 * Vh) + i;
        const uint4 a = STREAM ? ld_stream(pa) : __ldg(pa);
        const uint2 b = STREAM ? ld_stream(pb) : __ldg(pb);
        raw.w[0] = a.x; raw.w[1] = a.y; raw.w[2] = a.z; raw.w[3] = a.w; raw.w[4] = b.x; raw.w[5] = b.y;
    } else if constexpr (FMT == LINK_F32_12) {
        load_reals<float, 12, STREAM>(base, Vh, i, raw.r);
    } else if constexpr (FMT == LINK_F32_8) {
        load_reals<float, 8, STREAM>(base, Vh, i, raw.r);
    } else {
        float r[16];
        load_reals<float, 16, STREAM>(base, Vh, i, r);
#pragma unroll
        for (int k = 0; k < 16; k++) raw.r[k] = r[k];
        const float2 *tp = reinterpret_cast<const float2 *>(base + 64 * Vh) + i;
        float2 t = STREAM ? ld_stream(tp) : __ldg(tp);
        raw.r[16] = t.x;
        raw.r[17] = t.y;
    }
}

template <int FMT>
__device__ __forceinline__ void expand_link(const RawLink<FMT> &raw, typename LinkT<FMT>::T (&u)[18])
{
    if constexpr (FMT == LINK_F64_18 || FMT == LINK_F32_18) {
#pragma unroll
        for (int k = 0; k < 18; k++) u[k] = raw.r[k];
    } else if constexpr (FMT == LINK_I16_12) {
#pragma unroll
        for (int k = 0; k < 6; k++) unpack_i16(raw.w[k], u[2 * k], u[2 * k + 1]);
        reconstruct_row3(u);
    } else if constexpr (FMT == LINK_F32_8) {
        reconstruct8(raw.r, u);
    } else {
#pragma unroll
        for (int k = 0; k < 12; k++) u[k] = raw.r[k];
        reconstruct_row3(u);
    }
}

template <int FMT, bool STREAM = true>
__device__ __forceinline__ void load_link(const char *base, size_t Vh, size_t i, typename LinkT<FMT>::T (&u)[18])
{
    RawLink<FMT> raw;
    load_raw_link<FMT, STREAM>(base, Vh, i, raw);
    expand_link<FMT>(raw, u);
}

// ---- packed clover: per site 2 chiral blocks x (6 real diagonal + 15 complex strictly-lower entries,
// row-wise: (1,0),(2,0),(2,1),(3,0)...) = 72 reals.  Component index inside a block = 3*(s mod 2) + c.
// w = C v for one block; v, w are 6 complex = 12 reals; c = the block's 36 reals.
template <typename T>
__device__ __forceinline__ void clover_block_mul(const T *c, const T *v, T *w)
{
#pragma unroll
    for (int i = 0; i < 6; i++) {
        w[2 * i] = c[i] * v[2 * i];
        w[2 * i + 1] = c[i] * v[2 * i + 1];
    }
#pragma unroll
    for (int i = 1; i < 6; i++) {
#pragma unroll
        for (int j = 0; j < i; j++) {
            const int k = 6 + 2 * (i * (i - 1) / 2 + j);
            const T ar = c[k], ai = c[k + 1];
            // w_i += a v_j
            w[2 * i] = fma_(-ai, v[2 * j + 1], fma_(ar, v[2 * j], w[2 * i]));
            w[2 * i + 1] = fma_(ai, v[2 * j], fma_(ar, v[2 * j + 1], w[2 * i + 1]));
            // w_j += conj(a) v_i
            w[2 * j] = fma_(ai, v[2 * i + 1], fma_(ar, v[2 * i], w[2 * j]));
            w[2 * j + 1] = fma_(-ai, v[2 * i], fma_(ar, v[2 * i + 1], w[2 * j + 1]));
        }
    }
}

// The 36 packed reals of chiral block b of the clover field at site i; clov = [72/N chunks][Vh]
// H16: the field is stored in fp16, per block 4 chunks of 8 halfs + 1 chunk of 4 halfs (72 bytes), [block][chunk][Vh]
template <typename T, bool STREAM, bool H16>
__device__ __forceinline__ void load_clover_block(const void *clov, size_t Vh, size_t i, int b, T (&c)[36])
{
    typedef typename VT<T>::V V;
    constexpr int N = VT<T>::N;
    if constexpr (H16) {
        const char *base = reinterpret_cast<const char *>(clov) + (size_t)b * 72 * Vh;
#pragma unroll
        for (int k = 0; k < 4; k++) {
            const uint4 *p = reinterpret_cast<const uint4 *>(base + (size_t)k * 16 * Vh) + i;
            const uint4 q = STREAM ? ld_stream(p) : __ldg(p);
            unpack_h16(q.x, c[8 * k], c[8 * k + 1]);
            unpack_h16(q.y, c[8 * k + 2], c[8 * k + 3]);
            unpack_h16(q.z, c[8 * k + 4], c[8 * k + 5]);
            unpack_h16(q.w, c[8 * k + 6], c[8 * k + 7]);
        }
        const uint2 *p2 = reinterpret_cast<const uint2 *>(base + (size_t)64 * Vh) + i;
        const uint2 q2 = STREAM ? ld_stream(p2) : __ldg(p2);
        unpack_h16(q2.x, c[32], c[33]);
        unpack_h16(q2.y, c[34], c[35]);
    } else {
        load_reals<T, 36, STREAM>(reinterpret_cast<const V *>(clov) + (size_t)b * (36 / N) * Vh, Vh, i, c);
    }
}

// w = C(site i) v on the full 24-real spinor
template <typename T, bool STREAM = true, bool H16 = false>
__device__ __forceinline__ void clover_apply(const void *clov, size_t Vh, size_t i, const T (&v)[24], T (&w)[24])
{
#pragma unroll
    for (int b = 0; b < 2; b++) {
        T c[36];
        load_clover_block<T, STREAM, H16>(clov, Vh, i, b, c);
        clover_block_mul(c, &v[12 * b], &w[12 * b]);
    }
}

// Packed 36 reals of chiral block b of A from its 48-real form (CLOVER_G48_REALS in cola_internal.h):
//   block = 1 + [[G3, G1 - i G2], [G1 + i G2, -G3]],  G_j traceless Hermitian 3x3 as [d0, d1, l10, l20, l21]
template <typename T, bool STREAM>
__device__ __forceinline__ void load_clover_g48(const void *clov, size_t Vh, size_t i, int b, T (&c)[36])
{
    typedef typename VT<T>::V V;
    constexpr int N = VT<T>::N;
    T g[24];
    load_reals<T, 24, STREAM>(reinterpret_cast<const V *>(clov) + (size_t)b * (24 / N) * Vh, Vh, i, g);
    const T *G3 = g, *G1 = g + 8, *G2 = g + 16;
    const T one = 1, d32 = -(G3[0] + G3[1]);
    c[0] = one + G3[0]; c[1] = one + G3[1]; c[2] = one + d32;
    c[3] = one - G3[0]; c[4] = one - G3[1]; c[5] = one - d32;
    c[6] = G3[2]; c[7] = G3[3]; c[8] = G3[4]; c[9] = G3[5]; c[10] = G3[6]; c[11] = G3[7];       // (1,0) (2,0) (2,1)
    c[12] = G1[0]; c[13] = G2[0];                                                               // (3,0) = W_00, W = G1 + i G2
    c[14] = G1[2] + G2[3]; c[15] = G2[2] - G1[3];                                               // (3,1) = W_01 = conj(l10_1) + i conj(l10_2)
    c[16] = G1[4] + G2[5]; c[17] = G2[4] - G1[5];                                               // (3,2) = W_02
    c[18] = G1[2] - G2[3]; c[19] = G1[3] + G2[2];                                               // (4,0) = W_10 = l10_1 + i l10_2
    c[20] = G1[1]; c[21] = G2[1];                                                               // (4,1) = W_11
    c[22] = G1[6] + G2[7]; c[23] = G2[6] - G1[7];                                               // (4,2) = W_12
    c[24] = -G3[2]; c[25] = -G3[3];                                                             // (4,3) = -G3_10
    c[26] = G1[4] - G2[5]; c[27] = G1[5] + G2[4];                                               // (5,0) = W_20
    c[28] = G1[6] - G2[7]; c[29] = G1[7] + G2[6];                                               // (5,1) = W_21
    c[30] = -(G1[0] + G1[1]); c[31] = -(G2[0] + G2[1]);                                         // (5,2) = W_22
    c[32] = -G3[4]; c[33] = -G3[5]; c[34] = -G3[6]; c[35] = -G3[7];                             // (5,3) (5,4)
}

// w = A(site i) v with A in its 48-real form
template <typename T, bool STREAM = true>
__device__ __forceinline__ void clover_apply_g48(const void *clov, size_t Vh, size_t i, const T (&v)[24], T (&w)[24])
{
#pragma unroll
    for (int b = 0; b < 2; b++) {
        T c[36];
        load_clover_g48<T, STREAM>(clov, Vh, i, b, c);
        clover_block_mul(c, &v[12 * b], &w[12 * b]);
    }
}

// ---- deterministic reduction: warp shuffle -> shared -> per-block partial -> the last block to
// finish adds the partials in a fixed order.  All threads of the block must call it.
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ double block_sum(double v, double *sm /* >= 32 doubles */)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) sm[w] = v;
    __syncthreads();
    if (w == 0) {
        double t = lane < nw ? sm[lane] : 0.0;
        t = warp_sum(t);
        if (lane == 0) sm[0] = t;
    }
    __syncthreads();
    return sm[0];
}

// Workspace of one grid-wide reduction: per-block partials, then per-group partials, then per-group tickets.
// Blocks are grouped by REDUCE_GROUP consecutive block indices; the last block of a group to arrive adds the group's
// partials in index order, the last group to finish adds the group sums in index order.  Two short dependent steps
// instead of one block walking over every partial, and still bitwise deterministic (fixed order at each level).
// Returns true in thread 0 of the block that completes the reduction, with the grid-wide sum in *total.
// `counter` is the top-level ticket (self-resetting).  All threads of every block must call it.
__device__ __forceinline__ bool grid_sum_last(double v, const ReduceWs &ws, unsigned *counter, double *total)
{
    __shared__ double sm[33];
    __shared__ int stage;
    const unsigned group = blockIdx.x / REDUCE_GROUP;
    const unsigned ngroups = (gridDim.x + REDUCE_GROUP - 1) / REDUCE_GROUP;
    const unsigned first = group * REDUCE_GROUP;
    const unsigned gsize = min(REDUCE_GROUP, gridDim.x - first);
    double s = block_sum(v, sm);
    if (threadIdx.x == 0) {
        ws.partials[blockIdx.x] = s;
        __threadfence();
        stage = (atomicAdd(ws.gticket + group, 1u) == gsize - 1) ? 1 : 0;
    }
    __syncthreads();
    if (!stage) return false;
    __threadfence();
    double a = 0.0;
    for (unsigned k = threadIdx.x; k < gsize; k += blockDim.x) a += __ldcg(ws.partials + first + k);
    a = block_sum(a, sm);
    if (threadIdx.x == 0) {
        ws.gticket[group] = 0u;
        ws.gpart[group] = a;
        __threadfence();
        stage = (atomicAdd(counter, 1u) == ngroups - 1) ? 2 : 0;
    }
    __syncthreads();
    if (stage != 2) return false;
    __threadfence();
    a = 0.0;
    for (unsigned k = threadIdx.x; k < ngroups; k += blockDim.x) a += __ldcg(ws.gpart + k);
    a = block_sum(a, sm);
    if (threadIdx.x != 0) return false;
    *counter = 0u;
    *total = a;
    return true;
}

// The same for N values at once (component c uses partials + c*pstride, gpart + c*gstride; one ticket per group).
template <int N>
__device__ __forceinline__ bool grid_sum_last_n(const double (&v)[N], const ReduceWs &ws, unsigned *counter, double (&total)[N])
{
    __shared__ double sm[33];
    __shared__ int stage;
    static_assert(N <= REDUCE_MAXC, "too many reduction components");
    const unsigned group = blockIdx.x / REDUCE_GROUP;
    const unsigned ngroups = (gridDim.x + REDUCE_GROUP - 1) / REDUCE_GROUP;
    const unsigned first = group * REDUCE_GROUP;
    const unsigned gsize = min(REDUCE_GROUP, gridDim.x - first);
    double s[N];
#pragma unroll
    for (int c = 0; c < N; c++) s[c] = block_sum(v[c], sm);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int c = 0; c < N; c++) ws.partials[(size_t)c * ws.pstride + blockIdx.x] = s[c];
        __threadfence();
        stage = (atomicAdd(ws.gticket + group, 1u) == gsize - 1) ? 1 : 0;
    }
    __syncthreads();
    if (!stage) return false;
    __threadfence();
#pragma unroll
    for (int c = 0; c < N; c++) {
        double a = 0.0;
        for (unsigned k = threadIdx.x; k < gsize; k += blockDim.x) a += __ldcg(ws.partials + (size_t)c * ws.pstride + first + k);
        s[c] = block_sum(a, sm);
    }
    if (threadIdx.x == 0) {
        ws.gticket[group] = 0u;
#pragma unroll
        for (int c = 0; c < N; c++) ws.gpart[(size_t)c * ws.gstride + group] = s[c];
        __threadfence();
        stage = (atomicAdd(counter, 1u) == ngroups - 1) ? 2 : 0;
    }
    __syncthreads();
    if (stage != 2) return false;
    __threadfence();
#pragma unroll
    for (int c = 0; c < N; c++) {
        double a = 0.0;
        for (unsigned k = threadIdx.x; k < ngroups; k += blockDim.x) a += __ldcg(ws.gpart + (size_t)c * ws.gstride + k);
        s[c] = block_sum(a, sm);
    }
    if (threadIdx.x != 0) return false;
    *counter = 0u;
#pragma unroll
    for (int c = 0; c < N; c++) total[c] = s[c];
    return true;
}

__device__ __forceinline__ void grid_sum_finalize(double v, const ReduceWs &ws, unsigned *counter, double *result, bool accumulate = false)
{
    double a;
    if (grid_sum_last(v, ws, counter, &a)) *result = accumulate ? *result + a : a;
}

}  // namespace cola
