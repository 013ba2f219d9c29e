// cola_dslash_tile.cu -- the parity dslash family with the neighbour spinors STAGED IN SHARED MEMORY (BJ:ns: "shared-memory
// or TMA staging of neighbour half-spinors along the fastest-varying dimension").
//
// Why.  In the direct kernels (cola_dslash.cu) every thread fetches its 8 neighbour spinors through L1.  A thread block
// there is a run of 64 consecutive sites (a few x-rows of one z,t), so only the x and most of the y neighbours hit L1;
// the z and t neighbours come from L2 every time.  ncu: 0.95 GB of L2->L1 traffic per launch of the plain fp32 dslash
// at 32^3x64 against 0.58 GB of DRAM traffic -- 5800-6200 bytes per clock chip-wide, which is the ceiling of the
// L2-to-SM fabric (~6300 B/clk, B300_MICROARCH.md), not of HBM.  The kernels whose DRAM bytes are small (plain dslash,
// 16-bit fields, several right-hand sides) are bound there, and their 48 dependent LDG.128 per site expose L2 latency.
//
// How.  A block owns a 4-D tile of output sites, Xh x TY x TZ x TT in checkerboard coordinates (full rows in x, so the
// x neighbours wrap inside the row).  It copies the tile's input spinors and the six faces next to it (y-, y+, z-,
// z+, t-, t+) from global to shared memory with TMA bulk copies (cp.async.bulk, one per contiguous run of rows; an
// mbarrier counts the bytes), each input spinor ONCE per tile instead of once per use: 3.5-4 spinor loads per site
// instead of ~6 through L2.  (A first version issued one 16-byte cp.async per thread and chunk: +37 % executed
// instructions and, with L1 bypassed, 2x the expected L2->L1 bytes -- 20-28 % slower than the direct kernels.)  After
// the barrier every thread runs the 8 hops of its site reading neighbours with LDS.128; only the links (read exactly once,
// no reuse to exploit) still come from global memory, software-pipelined two hops ahead in registers and, with
// programmatic dependent launch, requested before the wait on the previous kernel (the gauge field is constant).
// The arithmetic of a site is the same sequence of calls as in the direct kernels (cola_hop.cuh): results are
// bit-identical (tests/test_gpu_sweep.py), only the summation order of the fused norm differs.
//
// fp32 and 16-bit formats only: the fp64 kernels are at the HBM roofline already and their tiles would need 2x the
// shared memory.
#include <string.h>

#include "cola_hop.cuh"

namespace cola {

namespace {

constexpr int TILE_MAX_THREADS = 256;
constexpr int TILE_STRIDE = 1024;   // shared-memory entries per 16-byte chunk plane (compile-time: LDS offsets become immediates)
#ifndef COLA_TILE_MINB
#define COLA_TILE_MINB 2
#endif

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");   // visible to the async (TMA) proxy
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    unsigned done;
    do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\nselp.u32 %0, 1, 0, p;\n}"
                     : "=r"(done)
                     : "r"(smem_u32(bar)), "r"(parity), "r"(2000u)   // suspend-time hint in ns: poll rarely
                     : "memory");
    } while (!done);
}
// TMA bulk copy (1-D, no tensor map): `bytes` (multiple of 16) from global to shared memory, completion counted on `bar`
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src), "r"(bytes),
                 "r"(smem_u32(bar))
                 : "memory");
}

template <typename T>
__device__ __forceinline__ void lds_spinor(const float4 *sm, const int stride, const int e, T (&psi)[24])
{
#pragma unroll
    for (int k = 0; k < 6; k++) {
        const float4 v = sm[k * stride + e];
        psi[4 * k] = v.x; psi[4 * k + 1] = v.y; psi[4 * k + 2] = v.z; psi[4 * k + 3] = v.w;
    }
}

// hop H = 2*MU + BACK: neighbour spinor from shared memory entry e, link from the raw buffer, which is then refilled with
// the link of hop H+2 (site li_next of gauge_next; nullptr: nothing left to load)
template <int FMT, int H, typename T>
__device__ __forceinline__ void hop_smem(const float4 *sm, const int stride, const int e, RawLink<FMT> &raw, const char *gauge_next, const size_t Vh,
                                         const int li_next, const T eta, const T s, T (&acc)[24])
{
    constexpr int MU = H >> 1;
    constexpr bool BACK = (H & 1) != 0;
    T psi[24], h[12], g[12], u[18];
    expand_link<FMT>(raw, u);
    if (H < 6) load_raw_link<FMT, true>(gauge_next, Vh, li_next, raw);
    lds_spinor(sm, stride, e, psi);
    project<MU>(psi, s, h);
    su3_mul<BACK>(u, h, g);
    reconstruct_accumulate<MU>(g, eta, s, acc);
}

template <int FMT, int XPAY, int POST>
__global__ void __launch_bounds__(TILE_MAX_THREADS, COLA_TILE_MINB) dslash_tile_kernel(const __grid_constant__ TileArgs ta)
{
    typedef typename LinkT<FMT>::T T;
    static_assert(sizeof(T) == 4, "the staged kernels are fp32 / 16-bit only");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint4 *smu = reinterpret_cast<uint4 *>(smem_raw);
    const float4 *smf = reinterpret_cast<const float4 *>(smem_raw);
    const DslashArgs &a = ta.d;
    const Geom &g = a.g;
    const size_t Vh = g.Vh;
    __shared__ __align__(8) unsigned long long mbar_storage;
    unsigned long long *mbar = &mbar_storage;
    if (threadIdx.x == 0) mbar_init(mbar, 1);
    pdl_trigger();
    __syncthreads();

    // tile origin (tiles ordered y fastest, then z, then t: the same time-slice-by-time-slice sweep as the direct kernels)
    const unsigned b = blockIdx.x;
    const unsigned q1 = ta.nby.div(b), by = b - q1 * ta.nby.d;
    const unsigned bt = ta.nbz.div(q1), bz = q1 - bt * ta.nbz.d;
    const int y0 = (int)by * ta.TY, z0 = (int)bz * ta.TZ, t0 = (int)bt * ta.TT;
    // this thread's site
    const unsigned l = threadIdx.x;
    const bool live = (int)l < ta.nthr;
    const unsigned lc = live ? l : 0u;
    const unsigned r1 = ta.dTX.div(lc), xh = lc - r1 * ta.dTX.d;
    const unsigned r2 = ta.dTY.div(r1), ly = r1 - r2 * ta.dTY.d;
    const unsigned lt = ta.dTZ.div(r2), lz = r2 - lt * ta.dTZ.d;
    const int y = y0 + (int)ly, z = z0 + (int)lz, t = t0 + (int)lt;
    const int sY = g.Xh, sZ = g.Xh * g.Y, sT = g.Xh * g.Y * g.Z;
    const int i = (int)xh + sY * y + sZ * z + sT * t;
    const int odd = (y + z + t + a.parity) & 1;     // x = 2*xh + odd

    // global cb indices of the sites whose links the backward hops read
    const int gxb = odd ? i : ((int)xh == 0 ? i + g.Xh - 1 : i - 1);
    const int gyb = (y == 0) ? i + (g.Y - 1) * sY : i - sY;
    const int gzb = (z == 0) ? i + (g.Z - 1) * sZ : i - sZ;
    const int gtb = (t == 0) ? i + (g.T - 1) * sT : i - sT;
    const size_t lb = link_bytes(FMT) * Vh;
    const char *gp = reinterpret_cast<const char *>(a.gauge_p);
    const char *gq = reinterpret_cast<const char *>(a.gauge_q);

    // the links of the first two hops do not depend on the previous kernel: request them before waiting for it
    RawLink<FMT> rawA, rawB;
    load_raw_link<FMT, true>(gp + 0 * lb, Vh, i, rawA);
    load_raw_link<FMT, true>(gq + 0 * lb, Vh, gxb, rawB);
    pdl_wait();
    if (a.skip && *a.skip) return;

    // ---- stage the tile's input spinors and its six faces with TMA bulk copies of whole x-y row groups.  With TX = Xh the
    // rows y0-1 .. y0+TY of fixed (z, t) are ONE contiguous run of (TY+2)*TX spinor chunks in the [chunk][site] layout
    // (three runs if the tile touches the y boundary of the lattice), and so is each z or t face at fixed t or z.
    // Shared-memory entries (16-byte chunk plane k at k * TILE_STRIDE):
    //   main(xh, ly, lz, lt) = xh + TX*((ly+1) + (TY+2)*(lz + TZ*lt)),  ly = -1 .. TY (the y faces are rows -1 and TY)
    //   zface(hi, lt)        = off_z + (hi*TT + lt)*TX*TY + xh + TX*ly
    //   tface(hi, lz)        = off_t + (hi*TZ + lz)*TX*TY + xh + TX*ly
    // Lane 0 of every warp issues the copies of the row groups dealt to its warp (72 copies per 256-site tile; a bulk
    // copy takes uniform registers and costs ~15 instructions of uniform-register traffic, so copies issued from divergent
    // lanes are serialised by the compiler, and all 72 issued by ONE lane take longer than the tile's arithmetic: 226 us
    // per launch against 114 us, ncu); the mbarrier is armed with the byte count of the whole tile; warp 0 waits on its
    // phase, the rest on the block barrier.
    const int TX = ta.TX, TY = ta.TY, TZ = ta.TZ, TT = ta.TT;
    const int rowsz = (TY + 2) * TX, face = TX * TY;
    if ((l & 31u) == 0u) {
        const int ym = y0 == 0 ? g.Y - 1 : y0 - 1, yp = y0 + TY == g.Y ? 0 : y0 + TY;
        const int zm = z0 == 0 ? g.Z - 1 : z0 - 1, zp = z0 + TZ == g.Z ? 0 : z0 + TZ;
        const int tm = t0 == 0 ? g.T - 1 : t0 - 1, tp = t0 + TT == g.T ? 0 : t0 + TT;
        const bool y_inside = y0 > 0 && y0 + TY < g.Y;
        const int nzt = TZ * TT, ngroups = nzt + 2 * TT + 2 * TZ;
        const uint4 *in = reinterpret_cast<const uint4 *>(a.in);
        if (l == 0) mbar_arrive_expect_tx(mbar, (unsigned)ta.nent * 96u);
        for (int gi = (int)(l >> 5); gi < ngroups; gi += (int)(blockDim.x >> 5)) {
            int zz, tt, ent;
            bool main_group = false;
            if (gi < nzt) {
                const int qt = (int)ta.dTZ.div((unsigned)gi), qz = gi - qt * TZ;
                zz = z0 + qz; tt = t0 + qt; ent = rowsz * gi;
                main_group = true;
            } else if (gi < nzt + 2 * TT) {
                const int q = gi - nzt, hi = q >= TT, qt = q - hi * TT;
                zz = hi ? zp : zm; tt = t0 + qt; ent = ta.off_z + q * face;
            } else {
                const int q = gi - nzt - 2 * TT, hi = q >= TZ, qz = q - hi * TZ;
                zz = z0 + qz; tt = hi ? tp : tm; ent = ta.off_t + q * face;
            }
            const size_t zt = (size_t)g.Y * ((size_t)zz + (size_t)g.Z * (size_t)tt);   // row index of (y = 0, zz, tt)
            uint4 *dst = smu + ent;
            if (!main_group) {
                const uint4 *src = in + (size_t)g.Xh * (zt + (size_t)y0);
#pragma unroll
                for (int k = 0; k < 6; k++) bulk_g2s(dst + k * TILE_STRIDE, src + (size_t)k * Vh, (unsigned)face * 16u, mbar);
            } else if (y_inside) {
                const uint4 *src = in + (size_t)g.Xh * (zt + (size_t)(y0 - 1));
#pragma unroll
                for (int k = 0; k < 6; k++) bulk_g2s(dst + k * TILE_STRIDE, src + (size_t)k * Vh, (unsigned)rowsz * 16u, mbar);
            } else {
                const uint4 *s0 = in + (size_t)g.Xh * (zt + (size_t)ym), *s1 = in + (size_t)g.Xh * (zt + (size_t)y0), *s2 = in + (size_t)g.Xh * (zt + (size_t)yp);
#pragma unroll
                for (int k = 0; k < 6; k++) {
                    bulk_g2s(dst + k * TILE_STRIDE, s0 + (size_t)k * Vh, (unsigned)TX * 16u, mbar);
                    bulk_g2s(dst + k * TILE_STRIDE + TX, s1 + (size_t)k * Vh, (unsigned)face * 16u, mbar);
                    bulk_g2s(dst + k * TILE_STRIDE + TX + face, s2 + (size_t)k * Vh, (unsigned)TX * 16u, mbar);
                }
            }
        }
    }

    // ---- shared-memory entries of the 8 neighbours and boundary signs (index arithmetic overlaps the copies)
    const int ec = (int)xh + TX * ((int)ly + 1 + (TY + 2) * ((int)lz + TZ * (int)lt));
    const int exf = odd ? ((int)xh + 1 == TX ? ec - (int)xh : ec + 1) : ec;
    const int exb = odd ? ec : ((int)xh == 0 ? ec + TX - 1 : ec - 1);
    const int fxy = (int)xh + TX * (int)ly;                      // position on a z or t face
    const int eyf = ec + TX, eyb = ec - TX;
    const int ezf = ((int)lz + 1 < TZ) ? ec + rowsz : ta.off_z + (TT + (int)lt) * face + fxy;
    const int ezb = ((int)lz > 0) ? ec - rowsz : ta.off_z + (int)lt * face + fxy;
    const int etf = ((int)lt + 1 < TT) ? ec + rowsz * TZ : ta.off_t + (TZ + (int)lz) * face + fxy;
    const int etb = ((int)lt > 0) ? ec - rowsz * TZ : ta.off_t + (int)lz * face + fxy;

    const bool cxf = odd && ((int)xh + 1 == g.Xh), cxb = !odd && ((int)xh == 0);
    const T one = 1;
    const T ex_f = (cxf && g.bc[0] < 0) ? -one : one, ex_b = (cxb && g.bc[0] < 0) ? -one : one;
    const T ey_f = (y + 1 == g.Y && g.bc[1] < 0) ? -one : one, ey_b = (y == 0 && g.bc[1] < 0) ? -one : one;
    const T ez_f = (z + 1 == g.Z && g.bc[2] < 0) ? -one : one, ez_b = (z == 0 && g.bc[2] < 0) ? -one : one;
    const T et_f = (t + 1 == g.T && g.bc[3] < 0) ? -one : one, et_b = (t == 0 && g.bc[3] < 0) ? -one : one;
    const T sf = (T)a.sgn, sb = -(T)a.sgn;   // forward: (1 + sgn*gamma), backward: (1 - sgn*gamma)

    // one warp polls the mbarrier (a polling loop executes instructions: eight spinning warps cost the other resident
    // tile 25 % of the issue slots, ncu), the others sleep on the block barrier
    if (l < 32u) mbar_wait(mbar, 0);
    __syncthreads();

    const bool want_norm = a.red.partials != nullptr;
    double nrm = 0.0;
    if (live) {
        T acc[24];
#pragma unroll
        for (int k = 0; k < 24; k++) acc[k] = 0;
        constexpr int st = TILE_STRIDE;
        hop_smem<FMT, 0>(smf, st, exf, rawA, gp + 1 * lb, Vh, i, ex_f, sf, acc);
        hop_smem<FMT, 1>(smf, st, exb, rawB, gq + 1 * lb, Vh, gyb, ex_b, sb, acc);
        hop_smem<FMT, 2>(smf, st, eyf, rawA, gp + 2 * lb, Vh, i, ey_f, sf, acc);
        hop_smem<FMT, 3>(smf, st, eyb, rawB, gq + 2 * lb, Vh, gzb, ey_b, sb, acc);
        hop_smem<FMT, 4>(smf, st, ezf, rawA, gp + 3 * lb, Vh, i, ez_f, sf, acc);
        hop_smem<FMT, 5>(smf, st, ezb, rawB, gq + 3 * lb, Vh, gtb, ez_b, sb, acc);
        hop_smem<FMT, 6>(smf, st, etf, rawA, nullptr, Vh, 0, et_f, sf, acc);
        hop_smem<FMT, 7>(smf, st, etb, rawB, nullptr, Vh, 0, et_b, sb, acc);
        nrm = dslash_epilogue<FMT, XPAY, POST, true>(a, i, acc, a.y, a.out, want_norm);
    }
    if (want_norm) grid_sum_finalize(nrm, a.red, a.counter, a.norm_out, a.norm_accumulate != 0);
}

template <int FMT, int XPAY, int POST>
cudaError_t launch_one(const TileArgs &ta, dim3 grid, dim3 block, size_t smem, cudaStream_t s)
{
    // The opt-in to > 48 KB of dynamic shared memory is an attribute of the function ON ONE DEVICE: keep the "done" flag
    // per instantiation and per device (contexts on different devices share this code).
    static bool configured[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        e = cudaFuncSetAttribute(dslash_tile_kernel<FMT, XPAY, POST>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    return launch_pdl_smem(dslash_tile_kernel<FMT, XPAY, POST>, grid, block, smem, s, ta);
}

template <int FMT>
cudaError_t launch_tile_fmt(const TileArgs &ta, cudaStream_t s)
{
    const DslashArgs &a = ta.d;
    const int xpay = a.y ? (a.clov_y ? (a.clov_y_g48 ? 3 : 2) : 1) : 0;
    const int post = a.clov_post ? 1 : 0;
    const dim3 grid((unsigned)ta.ntiles), block((unsigned)((ta.nthr + 31) / 32 * 32));
    const size_t smem = (size_t)TILE_STRIDE * 6 * 16;
    if (xpay == 0 && post == 0) return launch_one<FMT, 0, 0>(ta, grid, block, smem, s);
    if (xpay == 0 && post == 1) return launch_one<FMT, 0, 1>(ta, grid, block, smem, s);
    if (xpay == 1 && post == 0) return launch_one<FMT, 1, 0>(ta, grid, block, smem, s);
    if (xpay == 1 && post == 1) return launch_one<FMT, 1, 1>(ta, grid, block, smem, s);
    if (xpay == 2 && post == 0) return launch_one<FMT, 2, 0>(ta, grid, block, smem, s);
    if constexpr (FMT != LINK_I16_12)
        if (xpay == 3 && post == 0) return launch_one<FMT, 3, 0>(ta, grid, block, smem, s);
    return cudaErrorNotSupported;   // combination not instantiated: the caller falls back to the direct kernel
}

}  // namespace

// Tile of the staged kernels for a lattice: TX = Xh (full x rows), and the (TY, TZ, TT) dividing (Y, Z, T) with at most
// TILE_MAX_THREADS sites that stages the fewest input spinors per output site.  ok = 0 if no tile fits (Xh too large).
TileShape choose_tile(const Geom &g)
{
    TileShape best;
    memset(&best, 0, sizeof(best));
    if (g.Xh > TILE_MAX_THREADS) return best;
    double best_cost = 1e30;
    for (int ty = 1; ty <= g.Y; ty++) {
        if (g.Y % ty) continue;
        for (int tz = 1; tz <= g.Z; tz++) {
            if (g.Z % tz) continue;
            for (int tt = 1; tt <= g.T; tt++) {
                if (g.T % tt) continue;
                const int n = g.Xh * ty * tz * tt;
                if (n > TILE_MAX_THREADS) break;
                const int ent = n + 2 * g.Xh * (tz * tt + ty * tt + ty * tz);
                if (ent > TILE_STRIDE) continue;   // 96 KB of shared memory per tile: two tiles per SM
                // staged spinors per output site; idle lanes of the last warp count as sites that cost but do not produce
                const int lanes = (n + 31) / 32 * 32;
                const double cost = (double)ent / n * ((double)lanes / n);
                if (cost < best_cost - 1e-12 || (cost < best_cost + 1e-12 && n > best.nthr)) {
                    best_cost = cost;
                    best.ok = 1;
                    best.TY = ty; best.TZ = tz; best.TT = tt;
                    best.nthr = n;
                    best.nent = ent;
                }
            }
        }
    }
    return best;
}

cudaError_t launch_dslash_tile(int fmt, const DslashArgs &a, cudaStream_t s)
{
    const Geom &g = a.g;
    const TileShape sh = choose_tile(g);
    if (!sh.ok || fmt == LINK_F64_18) return cudaErrorNotSupported;
    TileArgs ta;
    memset(&ta, 0, sizeof(ta));
    ta.d = a;
    ta.TX = g.Xh; ta.TY = sh.TY; ta.TZ = sh.TZ; ta.TT = sh.TT;
    ta.nthr = sh.nthr;
    ta.nent = sh.nent;
    ta.stride = TILE_STRIDE;
    ta.ntiles = (g.Y / sh.TY) * (g.Z / sh.TZ) * (g.T / sh.TT);
    // a fused norm writes one partial per tile: small tiles (Xh small, extents with few divisors) can mean more tiles
    // than the reduction buffers have slots -- leave those launches to the direct kernel
    if (a.red.partials && (unsigned)ta.ntiles > a.red.pstride) return cudaErrorNotSupported;
    ta.off_z = sh.TZ * sh.TT * (sh.TY + 2) * g.Xh;
    ta.off_t = ta.off_z + 2 * sh.TT * g.Xh * sh.TY;
    ta.dTX = make_fastdiv((unsigned)g.Xh);
    ta.dTY = make_fastdiv((unsigned)sh.TY);
    ta.dTZ = make_fastdiv((unsigned)sh.TZ);
    ta.d1 = make_fastdiv(1u);
    ta.nby = make_fastdiv((unsigned)(g.Y / sh.TY));
    ta.nbz = make_fastdiv((unsigned)(g.Z / sh.TZ));
    switch (fmt) {
        case LINK_F32_18: return launch_tile_fmt<LINK_F32_18>(ta, s);
        case LINK_F32_12: return launch_tile_fmt<LINK_F32_12>(ta, s);
        case LINK_I16_12: return launch_tile_fmt<LINK_I16_12>(ta, s);
        case LINK_F32_8: return launch_tile_fmt<LINK_F32_8>(ta, s);
    }
    return cudaErrorNotSupported;
}

}  // namespace cola
