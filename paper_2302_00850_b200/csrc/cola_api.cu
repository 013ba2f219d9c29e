// cola_api.cu -- the C ABI of include/cola.h: context, workspace carving, gauge upload (H0-H2),
// operator entry points (H3-H8) and the CGNR / mixed-precision solvers (H9-H12).
#include <float.h>
#include <math.h>
#include <stdio.h>
#include <string.h>

#include "cola_internal.h"

using namespace cola;

struct cola_ctx {
    cola_params p;
    Geom g;
    size_t V, Vh;
    cudaStream_t stream;
    char err[512];
    int fmt32;
    // borrowed workspace, carved in cola_set_workspace
    char *ws;
    size_t ws_bytes;
    char *gauge64, *gauge32;        // [parity][mu][chunk][Vh]
    char *clovA64, *clovA32;        // [parity][chunk][Vh]
    char *clovI64, *clovI32;        // odd parity only
    char *gauge16, *clovA16, *clovI16;   // 16-bit copies for COLA_F32_H16 (same index structure)
    char *gauge8, *clovG32;         // COLA_F32_R8: links as 8 fp32 reals, A as its 48-real field-strength form (COLA_FEAT_R8)
    int r8_valid;                   // the 8-real links / 48-real A hold what the kernels assume (unitary links, traceless F)
    int compact;                    // bit 0: COLA_F32_R8 reads the 8-real links; bit 1: the fp32 operators read A in its 48-real form (cola_set_compact)
    unsigned features;              // COLA_FEAT_* parts of the workspace that are carved (cola_set_features)
    int h16_valid;                  // the 16-bit link copy holds what the kernels assume (12 reals of a unitary matrix)
    cola_prec inner_prec;           // operator precision of the running solve's fp32 iteration: COLA_F32, _H16 (mixed = 2) or _R8 (mixed = 3)
    double *hist;                   // HOST array of the running solve's residual history or nullptr (cola_cg_solve_history)
    int hist_len;
    int *upd_iters;                 // HOST array receiving the iterations at which reliable updates fired, or nullptr
    int upd_len;
    const char *defl_vecs;          // DEVICE eigenvectors of S^+S for the deflated start of the running solve, or nullptr
    const double *defl_evals;       // HOST
    int defl_n;
    // optional in-solve timing of the dominant kernel (cola_profile_kernel): event pairs around each launch of the
    // fused dslash + clover + xpay kernel of the inner precision
    int prof_on, prof_n;
    cudaEvent_t *prof_ev;           // 2 * PROF_MAX events, created on first use
    int prof_created;               // how many of them exist
    int staging;                    // 1: fp32 / 16-bit single-rhs kernels stage neighbour spinors in shared memory (cola_set_staging)
    size_t l2_budget;               // bytes of L2 the sweep order counts on for neighbour reuse (cola_set_l2_budget)
    char *tmp64, *tmp32;            // odd half-lattice temporaries of the Schur operator
    ReduceWs red;                   // deterministic-reduction buffers
    size_t red_blocks;              // max grid size of a reducing launch
    char *scratch;                  // solver vectors / staging
    size_t scratch_bytes;
    // owned
    Ctl *ctl;                       // device
    CtlB *ctlb;                     // device, inside the control block (BiCGStab scalars)
    unsigned long long *max_dev_bits;   // device (inside the same allocation)
    unsigned long long *min_pivot_key;  // device (inside the same allocation): see launch_clover_invert
    unsigned long long *min_u00_bits;   // device (inside the same allocation): min |U00|^2 over the links of the last upload
    double min_u00sq;
    double min_pivot;               // smallest Gauss-Jordan pivot of the 6x6 inverses of the last upload
    double *h_pinned;               // pinned host scalars
    HostStatus *h_status;           // mapped pinned host memory the device publishes the iteration status to
    HostStatus *d_status;           // device alias of h_status
    // multi-right-hand-side workspace (borrowed, cola_set_mrhs_workspace) and control state
    int m_nrhs;                     // capacity in right-hand sides (0: none)
    int m_solver;                   // the workspace also holds the batched solver's vectors
    char *m_tmp32;                  // [m_nrhs] odd half temporaries of the fp32 Schur operator
    char *m_r64;                    // [m_nrhs] fp64 half vectors: Schur temporary of the operator API; r of the batched solver
    char *m_rhs, *m_qs;             // [m_nrhs] fp64 half vectors: prepared sources, K x of the reliable updates
    char *m_x32, *m_r32, *m_p32, *m_q32;   // [m_nrhs] fp32 half vectors of the inner iteration
    char *m_rhat32;                 // [m_nrhs] fp32 shadow residuals of the batched BiCGStab
    CtlB *m_ctlb;                   // [MRHS_MAX] device scalars of the batched BiCGStab, one block per system
    HostStatus *m_statb;            // [MRHS_MAX] device: what each system's x/r update publishes
    double *m_tt;                   // [MRHS_MAX] device: |t_n|^2 as the multi-rhs operator reduces them
    HostStatus *h_statb;            // pinned host copy of m_statb (allocated on first use)
    double *m_partials;             // [m_nrhs][m_nsb]
    int m_nsb;
    CtlM *ctlm;                     // device, inside the control block
    HostStatusM *h_statusm, *d_statusm;   // mapped pinned host memory and its device alias
    cudaEvent_t ev0, ev1;
    int ready;
    double max_unitarity_dev;
    unsigned long long launches;
};

static thread_local char g_create_err[512] = "";
// message slot of calls that have no context (cola_create, cola_spinor_norm2_static): what cola_last_error(NULL) returns
void cola::set_thread_error(const char *msg) { snprintf(g_create_err, sizeof(g_create_err), "%s", msg); }
static const int PROF_MAX = 4096;   // launches timed per profiling window

static cola_status fail(cola_ctx *c, cola_status st, const char *fmt, const char *a = "", const char *b = "")
{
    char *dst = c ? c->err : g_create_err;
    snprintf(dst, 512, fmt, a, b);
    return st;
}

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e__ = (call);                                                                  \
        if (e__ != cudaSuccess) return fail(c, COLA_ECUDA, "%s: %s", #call, cudaGetErrorString(e__)); \
    } while (0)
#define ST(call)                          \
    do {                                  \
        cola_status s__ = (call);         \
        if (s__ != COLA_OK) return s__;   \
    } while (0)

static inline void cpu_relax()
{
#if defined(__x86_64__) || defined(__i386__)
    __builtin_ia32_pause();
#elif defined(__aarch64__)
    asm volatile("yield" ::: "memory");
#else
    __sync_synchronize();
#endif
}

static size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }
static size_t half_bytes(const cola_ctx *c, cola_prec prec) { return c->Vh * 24 * (prec == COLA_F64 ? 8 : 4); }   // COLA_F32_H16: fp32 spinors
// Solver scratch in units of one fp64 half-lattice spinor.  Even-odd solves use at most 9 slots (source 2, solution 2,
// prepared source 1, r 1, K x 1, four fp32 vectors 2), solves on M at most 12 (mixed: r 2, K x 2, four fp32 vectors 4).
// The *_host entry points need no more: the canonical source is staged where the solution will live and the canonical
// solution is written over the packed source once it is dead (cola_cg_solve_host).
static size_t scratch_half64(const cola_ctx *c) { return (c->features & COLA_FEAT_FULL_M) ? 12 : 9; }

struct Carve {
    size_t gauge64, gauge32, clovA64, clovA32, clovI64, clovI32, gauge16, clovA16, clovI16, gauge8, clovG32, tmp64, tmp32, partials, scratch, total;
};

static Carve carve(const cola_ctx *c)
{
    Carve k;
    size_t off = 0;
    const size_t Vh = c->Vh;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
    const size_t npar = (c->features & COLA_FEAT_FULL_M) ? 2 : 1;   // parities the fp32 / fp16 copies of A cover
    const size_t h16 = (c->features & COLA_FEAT_H16) ? 1 : 0;
    k.gauge64 = take(8 * 144 * Vh);
    k.gauge32 = take(8 * link_bytes(c->fmt32) * Vh);
    k.clovA64 = take(2 * 576 * Vh);         // fp64 A on both parities: the true residual is always |b - M x| on the full lattice
    k.clovA32 = take(((c->features & COLA_FEAT_A72) || !c->p.trace_sub ? 1 : 0) * npar * 288 * Vh);
    k.clovI64 = take(576 * Vh);
    k.clovI32 = take(288 * Vh);
    k.gauge16 = take(h16 * 8 * link_bytes(LINK_I16_12) * Vh);
    k.clovA16 = take(h16 * npar * CLOVER_H16_BYTES * Vh);
    k.clovI16 = take(h16 * CLOVER_H16_BYTES * Vh);
    const size_t r8 = (c->features & COLA_FEAT_R8) ? 1 : 0;
    k.gauge8 = take(r8 * 8 * link_bytes(LINK_F32_8) * Vh);
    k.clovG32 = take((c->p.trace_sub ? 1 : 0) * npar * CLOVER_G48_REALS * 4 * Vh);   // the form the fp32 kernels read A in (needs a traceless F)
    k.tmp64 = take(192 * Vh);
    k.tmp32 = take(96 * Vh);
    {
        size_t nb = dslash_grid_blocks(Vh);
        if (nb < (size_t)blas_max_blocks()) nb = (size_t)blas_max_blocks();
        k.partials = take(REDUCE_MAXC * (nb + reduce_groups(nb)) * sizeof(double) + reduce_groups(nb) * sizeof(unsigned));
    }
    k.scratch = take(scratch_half64(c) * 192 * Vh);
    k.total = off;
    return k;
}

extern "C" {

cola_status cola_create(cola_ctx **out, const cola_params *p)
{
    cola_ctx *c = nullptr;
    if (!out || !p) return fail(nullptr, COLA_EINVAL, "cola_create: NULL argument");
    *out = nullptr;
    for (int k = 0; k < 4; k++) {
        if (p->dims[k] < 2 || (p->dims[k] & 1)) return fail(nullptr, COLA_EINVAL, "cola_create: every extent must be even and >= 2");
        if (p->bc[k] != 1 && p->bc[k] != -1) return fail(nullptr, COLA_EINVAL, "cola_create: bc must be +1 or -1");
    }
    const double vol = (double)p->dims[0] * p->dims[1] * p->dims[2] * p->dims[3];
    if (vol / 2 > 2.0e9) return fail(nullptr, COLA_EINVAL, "cola_create: half volume exceeds 32-bit site indices");
    {
        cudaError_t e = cudaSetDevice(p->device);
        if (e != cudaSuccess) {
            cudaGetLastError();   // clear the (non-sticky) error so that it is not reported by a later launch of another context
            return fail(nullptr, COLA_ECUDA, "cudaSetDevice: %s", cudaGetErrorString(e));
        }
    }
    c = new cola_ctx();
    memset(c, 0, sizeof(*c));
    c->p = *p;
    c->g.X = p->dims[0]; c->g.Y = p->dims[1]; c->g.Z = p->dims[2]; c->g.T = p->dims[3];
    c->g.Xh = p->dims[0] / 2;
    c->g.dXh = make_fastdiv((unsigned)c->g.Xh);
    c->g.dY = make_fastdiv((unsigned)c->g.Y);
    c->g.dZ = make_fastdiv((unsigned)c->g.Z);
    c->V = (size_t)vol;
    c->Vh = c->V / 2;
    c->g.Vh = (int)c->Vh;
    for (int k = 0; k < 4; k++) c->g.bc[k] = p->bc[k];
    c->fmt32 = p->compress12 ? LINK_F32_12 : LINK_F32_18;
    c->l2_budget = (size_t)40 << 20;
    c->features = COLA_FEAT_ALL;
    c->compact = 3;
    c->inner_prec = COLA_F32;
    c->stream = (cudaStream_t)p->stream;
    char *blk = nullptr;
    cudaError_t e = cudaMalloc(&blk, 4096);
    if (e == cudaSuccess) e = cudaMemset(blk, 0, 4096);
    if (e == cudaSuccess) e = cudaHostAlloc(&c->h_pinned, 2048, cudaHostAllocMapped);
    if (e == cudaSuccess) e = cudaEventCreate(&c->ev0);
    if (e == cudaSuccess) e = cudaEventCreate(&c->ev1);
    if (e == cudaSuccess) {
        c->h_status = reinterpret_cast<HostStatus *>(reinterpret_cast<char *>(c->h_pinned) + 256);
        e = cudaHostGetDevicePointer(reinterpret_cast<void **>(&c->d_status), c->h_status, 0);
        c->h_statusm = reinterpret_cast<HostStatusM *>(reinterpret_cast<char *>(c->h_pinned) + 512);
        c->d_statusm = reinterpret_cast<HostStatusM *>(reinterpret_cast<char *>(c->d_status) + 256);
        static_assert(2 * sizeof(HostStatusM) <= 1536 && sizeof(Ctl) <= 512 && sizeof(CtlM) <= 1536, "control block layout");
    }
    if (e != cudaSuccess) {
        fail(nullptr, COLA_ECUDA, "cola_create: %s", cudaGetErrorString(e));
        if (blk) cudaFree(blk);
        if (c->h_pinned) cudaFreeHost(c->h_pinned);
        if (c->ev0) cudaEventDestroy(c->ev0);
        if (c->ev1) cudaEventDestroy(c->ev1);
        delete c;
        return COLA_ECUDA;
    }
    c->ctl = reinterpret_cast<Ctl *>(blk);
    c->ctlm = reinterpret_cast<CtlM *>(blk + 512);
    c->max_dev_bits = reinterpret_cast<unsigned long long *>(blk + 2048);
    c->min_pivot_key = reinterpret_cast<unsigned long long *>(blk + 2056);
    c->min_u00_bits = reinterpret_cast<unsigned long long *>(blk + 2064);
    c->ctlb = reinterpret_cast<CtlB *>(blk + 2304);
    static_assert(sizeof(CtlB) <= 512, "control block layout");
    *out = c;
    return COLA_OK;
}

cola_status cola_destroy(cola_ctx *c)
{
    if (!c) return COLA_OK;
    cudaSetDevice(c->p.device);
    cudaStreamSynchronize(c->stream);
    cudaFree(c->ctl);
    cudaFreeHost(c->h_pinned);
    if (c->h_statb) cudaFreeHost(c->h_statb);
    cudaEventDestroy(c->ev0);
    cudaEventDestroy(c->ev1);
    if (c->prof_ev) {
        for (int k = 0; k < c->prof_created; k++) cudaEventDestroy(c->prof_ev[k]);
        delete[] c->prof_ev;
    }
    delete c;
    return COLA_OK;
}

const char *cola_last_error(const cola_ctx *c) { return c ? c->err : g_create_err; }

cola_status cola_profile_kernel(cola_ctx *c, int enable)
{
    if (!c) return COLA_EINVAL;
    CK(cudaSetDevice(c->p.device));
    if (enable && c->prof_created < 2 * PROF_MAX) {
        if (!c->prof_ev) {
            c->prof_ev = new cudaEvent_t[2 * PROF_MAX];
            memset(c->prof_ev, 0, sizeof(cudaEvent_t) * 2 * PROF_MAX);
        }
        for (; c->prof_created < 2 * PROF_MAX; c->prof_created++) CK(cudaEventCreate(&c->prof_ev[c->prof_created]));
    }
    c->prof_on = enable ? 1 : 0;
    c->prof_n = 0;
    return COLA_OK;
}

cola_status cola_profile_result(cola_ctx *c, double *avg_ms, int *count, int *skipped)
{
    if (!c || !avg_ms || !count || !skipped) return COLA_EINVAL;
    *avg_ms = 0.0;
    *count = *skipped = 0;
    if (!c->prof_ev || c->prof_n == 0) return COLA_OK;
    CK(cudaSetDevice(c->p.device));
    CK(cudaStreamSynchronize(c->stream));
    float *ms = new float[2 * c->prof_n];
    for (int k = 0; k < c->prof_n; k++) {
        cudaError_t e = cudaEventElapsedTime(&ms[k], c->prof_ev[2 * k], c->prof_ev[2 * k + 1]);
        if (e != cudaSuccess) { delete[] ms; return fail(c, COLA_ECUDA, "cola_profile_result: %s", cudaGetErrorString(e)); }
        ms[c->prof_n + k] = ms[k];
    }
    // speculatively queued launches that found the flag raised return at once: they are not applications of the
    // operator.  Working launches are the large majority, so "well below the median" identifies the no-ops.
    float *sorted = ms + c->prof_n;
    for (int i = 1; i < c->prof_n; i++) {   // insertion sort: at most 4096 entries, once per window
        const float v = sorted[i];
        int j = i - 1;
        for (; j >= 0 && sorted[j] > v; j--) sorted[j + 1] = sorted[j];
        sorted[j + 1] = v;
    }
    const float median = sorted[c->prof_n / 2];
    double sum = 0.0;
    for (int k = 0; k < c->prof_n; k++) {
        if (ms[k] < 0.25f * median) (*skipped)++;
        else { sum += ms[k]; (*count)++; }
    }
    delete[] ms;
    if (*count) *avg_ms = sum / *count;
    c->prof_n = 0;
    return COLA_OK;
}

cola_status cola_set_l2_budget(cola_ctx *c, size_t bytes)
{
    if (!c) return COLA_EINVAL;
    c->l2_budget = bytes ? bytes : ((size_t)40 << 20);
    return COLA_OK;
}

cola_status cola_set_features(cola_ctx *c, unsigned features)
{
    if (!c) return COLA_EINVAL;
    if (features & ~(unsigned)COLA_FEAT_ALL) return fail(c, COLA_EINVAL, "cola_set_features: unknown feature bit");
    c->features = features;
    c->ws = nullptr;      // the carving changes: the workspace has to be lent again
    c->ws_bytes = 0;
    c->ready = 0;
    return COLA_OK;
}

cola_status cola_set_compact(cola_ctx *c, int mask)
{
    if (!c) return COLA_EINVAL;
    if (mask < 0 || mask > 3) return fail(c, COLA_EINVAL, "cola_set_compact: mask must be 0..3");
    c->compact = mask;
    return COLA_OK;
}

cola_status cola_set_staging(cola_ctx *c, int mode)
{
    if (!c) return COLA_EINVAL;
    if (mode < 0 || mode > 1) return fail(c, COLA_EINVAL, "cola_set_staging: mode must be 0 or 1");
    c->staging = mode;
    return COLA_OK;
}

cola_status cola_set_stream(cola_ctx *c, void *stream)
{
    if (!c) return COLA_EINVAL;
    c->stream = (cudaStream_t)stream;
    return COLA_OK;
}

size_t cola_spinor_bytes(const cola_ctx *c, cola_prec prec, int full)
{
    if (!c) return 0;
    return half_bytes(c, prec) * (full ? 2 : 1);
}

size_t cola_workspace_bytes(const cola_ctx *c) { return c ? carve(c).total : 0; }

cola_status cola_set_workspace(cola_ctx *c, void *dev_ptr, size_t bytes)
{
    if (!c) return COLA_EINVAL;
    c->ready = 0;
    if (!dev_ptr || ((uintptr_t)dev_ptr & 255)) return fail(c, COLA_EINVAL, "cola_set_workspace: pointer must be non-NULL and 256-byte aligned");
    const Carve k = carve(c);
    if (bytes < k.total) return fail(c, COLA_ENOMEM, "cola_set_workspace: workspace smaller than cola_workspace_bytes()");
    c->ws = (char *)dev_ptr;
    c->ws_bytes = bytes;
    c->gauge64 = c->ws + k.gauge64; c->gauge32 = c->ws + k.gauge32;
    c->clovA64 = c->ws + k.clovA64; c->clovA32 = c->ws + k.clovA32;
    c->clovI64 = c->ws + k.clovI64; c->clovI32 = c->ws + k.clovI32;
    c->gauge16 = c->ws + k.gauge16; c->clovA16 = c->ws + k.clovA16; c->clovI16 = c->ws + k.clovI16;
    c->tmp64 = c->ws + k.tmp64; c->tmp32 = c->ws + k.tmp32;
    {
        size_t nb = dslash_grid_blocks(c->Vh);
        if (nb < (size_t)blas_max_blocks()) nb = (size_t)blas_max_blocks();
        c->red_blocks = nb;
        c->red.partials = (double *)(c->ws + k.partials);
        c->red.pstride = (unsigned)nb;
        c->red.gstride = (unsigned)reduce_groups(nb);
        c->red.gpart = c->red.partials + REDUCE_MAXC * nb;
        c->red.gticket = (unsigned *)(c->red.gpart + REDUCE_MAXC * reduce_groups(nb));
        cudaError_t e = cudaMemsetAsync(c->red.gticket, 0, reduce_groups(nb) * sizeof(unsigned), c->stream);
        if (e != cudaSuccess) return fail(c, COLA_ECUDA, "cola_set_workspace: %s", cudaGetErrorString(e));
    }
    c->scratch = c->ws + k.scratch;
    c->scratch_bytes = scratch_half64(c) * 192 * c->Vh;
    if (!(c->features & COLA_FEAT_H16)) c->gauge16 = c->clovA16 = c->clovI16 = nullptr;
    c->gauge8 = (c->features & COLA_FEAT_R8) ? c->ws + k.gauge8 : nullptr;
    c->clovG32 = c->p.trace_sub ? c->ws + k.clovG32 : nullptr;
    if (!((c->features & COLA_FEAT_A72) || !c->p.trace_sub)) c->clovA32 = nullptr;
    return COLA_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// internal helpers
// ------------------------------------------------------------------------------------------------
static cola_status need_ready(cola_ctx *c, const char *who)
{
    if (!c) return COLA_EINVAL;
    if (!c->ws) return fail(c, COLA_ENOTREADY, "%s: no workspace (call cola_set_workspace)", who);
    if (!c->ready) return fail(c, COLA_ENOTREADY, "%s: no gauge field (call cola_gauge_upload)", who);
    return COLA_OK;
}

static bool r8_links(const cola_ctx *c, cola_prec prec) { return prec == COLA_F32_R8 && (c->compact & 1); }
// the fp32 operators (COLA_F32, COLA_F32_R8) read A in its 48-real form unless told otherwise (or F has a trace)
static bool r8_clover(const cola_ctx *c, cola_prec prec) { return (prec == COLA_F32_R8 || prec == COLA_F32) && c->clovG32 && ((c->compact & 2) || !c->clovA32); }
static int fmt_of(const cola_ctx *c, cola_prec prec)
{
    if (r8_links(c, prec)) return (int)LINK_F32_8;
    return prec == COLA_F64 ? (int)LINK_F64_18 : (prec == COLA_F32_H16 ? (int)LINK_I16_12 : c->fmt32);
}
static char *gauge_of(const cola_ctx *c, cola_prec prec, int parity)
{
    if (prec == COLA_F64) return c->gauge64 + (size_t)parity * 4 * 144 * c->Vh;
    if (prec == COLA_F32_H16) return c->gauge16 + (size_t)parity * 4 * link_bytes(LINK_I16_12) * c->Vh;
    if (r8_links(c, prec)) return c->gauge8 + (size_t)parity * 4 * link_bytes(LINK_F32_8) * c->Vh;
    return c->gauge32 + (size_t)parity * 4 * link_bytes(c->fmt32) * c->Vh;
}
static char *clovA_of(const cola_ctx *c, cola_prec prec, int parity)
{
    if (prec == COLA_F64) return c->clovA64 + (size_t)parity * 576 * c->Vh;
    if (prec == COLA_F32_H16) return c->clovA16 + (size_t)parity * CLOVER_H16_BYTES * c->Vh;
    if (r8_clover(c, prec)) return c->clovG32 + (size_t)parity * CLOVER_G48_REALS * 4 * c->Vh;
    return c->clovA32 + (size_t)parity * 288 * c->Vh;
}
static char *clovI_of(const cola_ctx *c, cola_prec prec) { return prec == COLA_F64 ? c->clovI64 : (prec == COLA_F32_H16 ? c->clovI16 : c->clovI32); }
static char *tmp_of(const cola_ctx *c, cola_prec prec) { return prec == COLA_F64 ? c->tmp64 : c->tmp32; }

// Is the operator of precision `prec` available with the carved features / the uploaded links?  uses_A: the launch
// reads A on `parity` (the fp32 / fp16 copies of A_oo exist only with COLA_FEAT_FULL_M).
static cola_status check_prec(cola_ctx *c, cola_prec prec, int parity, int uses_A)
{
    if ((int)prec < 0 || (int)prec > (int)COLA_F32_R8) return fail(c, COLA_EINVAL, "unknown cola_prec");
    if (prec == COLA_F32_R8) {
        if (!(c->features & COLA_FEAT_R8)) return fail(c, COLA_EINVAL, "COLA_F32_R8 / mixed = 3 need COLA_FEAT_R8 (cola_set_features)");
        if (!c->r8_valid)
            return fail(c, COLA_EINVAL, "COLA_F32_R8 / mixed = 3: needs links unitary to 1e-10 with every |U00| >= 0.1 (8-real parametrisation of SU(3); cola_gauge_info_r8)");
    }
    if (prec == COLA_F32_H16) {
        if (!(c->features & COLA_FEAT_H16)) return fail(c, COLA_EINVAL, "COLA_F32_H16 / mixed = 2 need COLA_FEAT_H16 (cola_set_features)");
        if (!c->h16_valid)
            return fail(c, COLA_EINVAL, "COLA_F32_H16 / mixed = 2: the uploaded links are not unitary to 1e-10, so their 16-bit copy (12 reals, third row rebuilt) is wrong");
    }
    if (prec != COLA_F64 && uses_A && parity == 1 && !(c->features & COLA_FEAT_FULL_M))
        return fail(c, COLA_EINVAL, "the fp32 operator on the full lattice needs COLA_FEAT_FULL_M (cola_set_features)");
    return COLA_OK;
}

// out_p = [post] ( [A] y + coef * D_{p,1-p} in ), optional |out|^2 -> norm_out
static cola_status dslash(cola_ctx *c, cola_prec prec, int parity, int dagger, const void *in, void *out, const void *y, int clov_on_y,
                          double coef, int post_inv, double *norm_out, int norm_accumulate, const int *skip = nullptr, double *dot_out = nullptr)
{
    ST(check_prec(c, prec, parity, (y && clov_on_y) ? 1 : 0));
    DslashArgs a;
    memset(&a, 0, sizeof(a));
    a.g = c->g;
    a.in = in;
    a.out = out;
    a.gauge_p = gauge_of(c, prec, parity);
    a.gauge_q = gauge_of(c, prec, 1 - parity);
    a.y = y;
    a.clov_y = (y && clov_on_y) ? clovA_of(c, prec, parity) : nullptr;
    a.clov_y_g48 = (a.clov_y && r8_clover(c, prec)) ? 1 : 0;
    a.clov_post = post_inv ? clovI_of(c, prec) : nullptr;
    a.coef = coef;
    a.sgn = dagger ? +1.0 : -1.0;
    a.parity = parity;
    a.skip = skip;
    a.sweep = make_sweep(c->g, choose_zband(c->g.Xh * c->g.Y, c->g.Z, prec == COLA_F64 ? 192 : 96, c->l2_budget, 1));
    if (norm_out) {
        a.red = c->red;
        a.counter = &c->ctl->counter[0];
        a.norm_out = norm_out;
        a.norm_accumulate = norm_accumulate;
        a.dot_out = y ? dot_out : nullptr;     // <out, y>, fused with the norm (direct kernels only)
    }
    if (post_inv && parity != 1) return fail(c, COLA_EINVAL, "internal: A^-1 is stored on the odd parity only");
    const bool timed = c->prof_on && c->prof_created == 2 * PROF_MAX && c->prof_n < PROF_MAX && prec != COLA_F64 && a.clov_y;   // Schur kernel 2 / M of the inner precision
    if (timed) CK(cudaEventRecord(c->prof_ev[2 * c->prof_n], c->stream));
    cudaError_t le = (c->staging && !a.dot_out) ? launch_dslash_tile(fmt_of(c, prec), a, c->stream) : cudaErrorNotSupported;
    if (le == cudaErrorNotSupported) le = launch_dslash(fmt_of(c, prec), a, c->stream);
    CK(le);
    if (timed) {
        CK(cudaEventRecord(c->prof_ev[2 * c->prof_n + 1], c->stream));
        c->prof_n++;
    }
    c->launches++;
    return COLA_OK;
}

// out_e = S in_e  (2 launches; norm of the result optional)
static cola_status schur(cola_ctx *c, cola_prec prec, int dagger, const void *in_e, void *out_e, double *norm_out, const int *skip = nullptr,
                         double *dot_out = nullptr)   // dot_out (with norm_out): <S in, in>
{
    const double k = c->p.kappa;
    ST(dslash(c, prec, 1, dagger, in_e, tmp_of(c, prec), nullptr, 0, 0.0, 1, nullptr, 0, skip));          // t_o = A_oo^-1 D_oe x_e
    ST(dslash(c, prec, 0, dagger, tmp_of(c, prec), out_e, in_e, 1, -k * k, 0, norm_out, 0, skip, dot_out));   // A_ee x_e - k^2 D_eo t_o
    return COLA_OK;
}

// out = M in on the full lattice (2 launches)
static cola_status fmatrix(cola_ctx *c, cola_prec prec, int dagger, const void *in, void *out, double *norm_out, const int *skip = nullptr)
{
    const size_t hb = half_bytes(c, prec);
    const char *in_e = (const char *)in, *in_o = in_e + hb;
    char *out_e = (char *)out, *out_o = out_e + hb;
    ST(dslash(c, prec, 0, dagger, in_o, out_e, in_e, 1, -c->p.kappa, 0, norm_out, 0, skip));
    ST(dslash(c, prec, 1, dagger, in_e, out_o, in_o, 1, -c->p.kappa, 0, norm_out, 1, skip));
    return COLA_OK;
}

static cola_status read_scalar(cola_ctx *c, const double *dev, double *host)
{
    CK(cudaMemcpyAsync(c->h_pinned, dev, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    *host = c->h_pinned[0];
    return COLA_OK;
}

static cola_status norm2(cola_ctx *c, cola_prec prec, const void *v, size_t n_sites, double *dev_out)
{
    CK(launch_norm2(prec, v, n_sites, c->red, &c->ctl->counter[2], dev_out, c->stream));
    c->launches++;
    return COLA_OK;
}

// ------------------------------------------------------------------------------------------------
// gauge upload (H0-H2)
// ------------------------------------------------------------------------------------------------
static cola_status gauge_finish(cola_ctx *c)
{
    unsigned long long bits = 0;
    CK(cudaMemcpyAsync(&bits, c->max_dev_bits, sizeof(bits), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    memcpy(&c->max_unitarity_dev, &bits, sizeof(double));
    CK(cudaMemcpyAsync(&bits, c->min_u00_bits, sizeof(bits), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    memcpy(&c->min_u00sq, &bits, sizeof(double));
    if (c->p.compress12 && !(c->max_unitarity_dev <= 1e-10))
        return fail(c, COLA_EINVAL, "cola_gauge_upload: links are not unitary to 1e-10; 12-real compression would be wrong");
    // the 16-bit copy stores rows 1 and 2 clamped to [-1, 1] and rebuilds row 3: only right for unitary links
    c->h16_valid = (c->features & COLA_FEAT_H16) && c->max_unitarity_dev <= 1e-10;
    c->r8_valid = (c->features & COLA_FEAT_R8) && c->max_unitarity_dev <= 1e-10 && c->min_u00sq >= R8_MIN_U00SQ;
    CK(launch_clover_build(c->g, c->gauge64, c->p.kappa * c->p.csw, c->p.trace_sub, c->clovA64, c->clovA32, (c->features & COLA_FEAT_FULL_M) ? 2 : 1,
                           c->clovA16, c->clovG32, c->stream));
    CK(cudaMemsetAsync(c->min_pivot_key, 0xff, sizeof(unsigned long long), c->stream));
    CK(launch_clover_invert(c->g, c->clovA64 + 576 * c->Vh, c->clovI64, c->clovI32, c->clovI16, c->min_pivot_key, c->stream));
    c->launches += 2;
    unsigned long long key = 0;
    CK(cudaMemcpyAsync(&key, c->min_pivot_key, sizeof(key), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    c->min_pivot = pivot_from_key(key);
    if (!(c->min_pivot > 0.0))
        return fail(c, COLA_EINVAL, "cola_gauge_upload: a 6x6 clover block on the odd parity is not positive definite (pivot <= 0): kappa*csw too large for these links");
    c->ready = 1;
    return COLA_OK;
}

static cola_status gauge_upload_impl(cola_ctx *c, const double *links, int on_host)
{
    if (!c) return COLA_EINVAL;
    if (!links) return fail(c, COLA_EINVAL, "cola_gauge_upload: NULL links");
    if (!c->ws) return fail(c, COLA_ENOTREADY, "cola_gauge_upload: no workspace (call cola_set_workspace)");
    CK(cudaSetDevice(c->p.device));
    c->ready = 0;
    CK(cudaMemsetAsync(c->max_dev_bits, 0, sizeof(unsigned long long), c->stream));
    CK(cudaMemsetAsync(c->min_u00_bits, 0x7f, sizeof(unsigned long long), c->stream));   // 0x7f7f...: a huge positive double
    if (!on_host) {
        CK(launch_gauge_reorder(c->g, links, 0, (long)c->V, c->gauge64, c->gauge32, c->fmt32, c->gauge16, c->gauge8, c->max_dev_bits, c->min_u00_bits, c->stream));
        c->launches++;
        return gauge_finish(c);
    }
    const size_t per_site = 4 * 18 * sizeof(double);
    size_t chunk_sites = c->scratch_bytes / per_site;
    if (chunk_sites > c->V) chunk_sites = c->V;
    for (size_t lo = 0; lo < c->V; lo += chunk_sites) {
        const size_t n = (c->V - lo < chunk_sites) ? c->V - lo : chunk_sites;
        CK(cudaMemcpyAsync(c->scratch, links + lo * 72, n * per_site, cudaMemcpyHostToDevice, c->stream));
        CK(launch_gauge_reorder(c->g, (const double *)c->scratch, (long)lo, (long)n, c->gauge64, c->gauge32, c->fmt32, c->gauge16, c->gauge8, c->max_dev_bits, c->min_u00_bits, c->stream));
        c->launches++;
    }
    return gauge_finish(c);
}

// ------------------------------------------------------------------------------------------------
// solvers (H9-H12)
// ------------------------------------------------------------------------------------------------
namespace {

struct System {            // K x = rhs on n_sites sites; K = S (even_odd) or M
    int even_odd;
    size_t n_sites;
};

cola_status apply_K(cola_ctx *c, const System &sy, cola_prec prec, int dagger, const void *in, void *out, double *norm_out, const int *skip = nullptr,
                    double *dot_out = nullptr)   // Schur system only: <K in, in> next to |K in|^2
{
    // the inner fp32 iteration of a mixed = 2 / 3 solve reads the 16-bit / compact fields (same fp32 vectors)
    const cola_prec op = (prec == COLA_F32) ? c->inner_prec : prec;
    return sy.even_odd ? schur(c, op, dagger, in, out, norm_out, skip, dot_out) : fmatrix(c, op, dagger, in, out, norm_out, skip);
}

// (re)arm the device-side decision state: rmax2, target2, delta2, flag = 0, iters
cola_status set_decision_state(cola_ctx *c, double rmax2, double target2, double delta2, int iters)
{
    struct { double rmax2, target2, delta2; int flag, iters; } st = {rmax2, target2, delta2, 0, iters};
    static_assert(sizeof(st) == 32, "decision block layout");
    static_assert(offsetof(Ctl, iters) - offsetof(Ctl, rmax2) == 28, "decision block layout");
    // pageable source: the runtime stages it before returning, so the stack buffer may die
    CK(cudaMemcpyAsync(&c->ctl->rmax2, &st, sizeof(st), cudaMemcpyHostToDevice, c->stream));
    return COLA_OK;
}

// Wait until iteration k's r_update has published its status (slot k & 1, sequence number k + 1).  The device
// writes straight into mapped pinned memory, so this is a poll on host memory, not a stream synchronisation;
// the stream is queried now and then so that a faulted kernel cannot hang the caller.
cola_status wait_status(cola_ctx *c, int k, HostStatus *out)
{
    volatile HostStatus *m = c->h_status + (k & 1);
    for (unsigned long spins = 0;; spins++) {
        if (m->iters == k + 1) break;
        if ((spins & 0xfff) == 0xfff) {
            cudaError_t e = cudaStreamQuery(c->stream);
            if (e == cudaSuccess) {
                if (m->iters == k + 1) break;
                return fail(c, COLA_ECUDA, "cola_cg_solve: the stream drained without iteration status (internal error)");
            }
            if (e != cudaErrorNotReady) return fail(c, COLA_ECUDA, "cola_cg_solve: %s", cudaGetErrorString(e));
        }
        cpu_relax();
    }
    __sync_synchronize();
    out->rr = m->rr;
    out->flag = m->flag;
    out->iters = m->iters;
    return COLA_OK;
}

// iteration k, first half:  q = K p (|q|^2),  r -= alpha q (|r|^2, decision, status -> mapped host slot k & 1)
cola_status first_half(cola_ctx *c, const System &sy, cola_prec P, int k, char *ri, char *pi, char *qi)
{
    Ctl *ctl = c->ctl;
    ST(apply_K(c, sy, P, 0, pi, qi, &ctl->qq, &ctl->flag));
    CK(launch_r_update(P, ri, qi, ctl, k & 1, k + 1, &ctl->flag, c->d_status + (k & 1), sy.n_sites, c->red, c->stream));
    c->launches++;
    return COLA_OK;
}

// iteration k, second half:  s = K^+ r (|s|^2),  x += alpha p (do_x),  p = s + beta p
cola_status second_half(cola_ctx *c, const System &sy, cola_prec P, int k, int do_x, char *xi, char *ri, char *pi, char *qi)
{
    Ctl *ctl = c->ctl;
    ST(apply_K(c, sy, P, 1, ri, qi, &ctl->gam[(k & 1) ^ 1], &ctl->flag));
    CK(launch_xp_update(P, xi, pi, qi, ctl, k & 1, do_x, 1, &ctl->flag, sy.n_sites, c->stream));
    c->launches++;
    return COLA_OK;
}

size_t vec_bytes(const cola_ctx *c, const System &sy, cola_prec prec) { return half_bytes(c, prec) * (sy.even_odd ? 1 : 2); }

// out64 = a*A + b*B with an optional fp32 copy; per half lattice because the fp64<->fp32 chunk
// pairing of the internal layout is per half
cola_status axpby64(cola_ctx *c, const System &sy, void *out64, double a, const void *A, double b, const void *B, void *out32)
{
    const int nh = sy.even_odd ? 1 : 2;
    for (int h = 0; h < nh; h++) {
        const size_t o64 = h * half_bytes(c, COLA_F64), o32 = h * half_bytes(c, COLA_F32);
        CK(launch_axpby64((char *)out64 + o64, a, (const char *)A + o64, b, B ? (const char *)B + o64 : nullptr,
                          out32 ? (char *)out32 + o32 : nullptr, c->Vh, nullptr, nullptr, nullptr, c->stream));
        c->launches++;
    }
    return COLA_OK;
}

}  // namespace

static cola_status solve_bicgstab_impl(cola_ctx *c, const cola_solve_params *sp, const void *b_canon_dev, void *x_canon_dev, cola_solve_info *info);

static cola_status solve_impl(cola_ctx *c, const cola_solve_params *sp, const void *b_canon_dev, void *x_canon_dev, cola_solve_info *info)
{
    if (c && sp && sp->method == COLA_BICGSTAB) return solve_bicgstab_impl(c, sp, b_canon_dev, x_canon_dev, info);
    if (c && sp && sp->method != COLA_CGNR) return fail(c, COLA_EINVAL, "cola_cg_solve: unknown method");
    ST(need_ready(c, "cola_cg_solve"));
    if (!sp || !b_canon_dev || !x_canon_dev || !info) return fail(c, COLA_EINVAL, "cola_cg_solve: NULL argument");
    if (!(sp->tol > 0) || sp->max_iter < 1) return fail(c, COLA_EINVAL, "cola_cg_solve: tol must be > 0 and max_iter >= 1");
    CK(cudaSetDevice(c->p.device));
    memset(info, 0, sizeof(*info));
    if (sp->mixed < 0 || sp->mixed > 3) return fail(c, COLA_EINVAL, "cola_cg_solve: mixed must be 0, 1, 2 or 3");
    if (sp->mixed == 2) ST(check_prec(c, COLA_F32_H16, 0, 0));
    if (sp->mixed == 3) ST(check_prec(c, COLA_F32_R8, 0, 0));
    if (!sp->even_odd && !(c->features & COLA_FEAT_FULL_M))
        return fail(c, COLA_EINVAL, "cola_cg_solve: even_odd = 0 (CGNR on M) needs COLA_FEAT_FULL_M (cola_set_features)");
    c->inner_prec = sp->mixed == 2 ? COLA_F32_H16 : (sp->mixed == 3 ? COLA_F32_R8 : COLA_F32);
    const double delta = sp->delta > 0 ? sp->delta : 0.1;
    const double kappa = c->p.kappa;
    const size_t h64 = half_bytes(c, COLA_F64), h32 = half_bytes(c, COLA_F32);
    System sy;
    sy.even_odd = sp->even_odd ? 1 : 0;
    sy.n_sites = sy.even_odd ? c->Vh : c->V;
    const size_t nv64 = vec_bytes(c, sy, COLA_F64), nv32 = vec_bytes(c, sy, COLA_F32);
    const double flops_K = sy.even_odd ? 3696.0 * (double)c->Vh : 1872.0 * (double)c->V;
    double flops = 0.0;

    // scratch carving (units of fp64 half vectors; SCRATCH_HALF64 = 12 covers the worst case)
    char *sc = c->scratch;
    char *B = sc; sc += 2 * h64;          // packed source, full lattice
    char *X = sc; sc += 2 * h64;          // solution, full lattice (x_e is its even half)
    char *rhs, *r, *p = nullptr, *qs;
    char *x32 = nullptr, *r32 = nullptr, *p32 = nullptr, *qs32 = nullptr;
    if (sy.even_odd) { rhs = sc; sc += h64; } else rhs = B;
    r = sc; sc += nv64;
    qs = sc; sc += nv64;
    if (!sp->mixed) { p = sc; sc += nv64; }
    else {
        x32 = sc; sc += nv32;
        r32 = sc; sc += nv32;
        p32 = sc; sc += nv32;
        qs32 = sc; sc += nv32;
    }
    if ((size_t)(sc - c->scratch) > c->scratch_bytes) return fail(c, COLA_ENOMEM, "cola_cg_solve: internal scratch too small");
    char *xsol = X;                       // x of the iterated system (even half of X, or all of X)

    Ctl *ctl = c->ctl;
    CK(cudaEventRecord(c->ev0, c->stream));
    CK(launch_spinor_pack(COLA_F64, c->g, b_canon_dev, B, c->stream));
    c->launches++;
    double bb = 0.0;
    ST(norm2(c, COLA_F64, B, c->V, &ctl->aux[2]));
    ST(read_scalar(c, &ctl->aux[2], &bb));
    if (!(bb <= DBL_MAX)) return fail(c, COLA_EINVAL, "cola_cg_solve: the source contains NaN or Inf");
    CK(cudaMemsetAsync(X, 0, 2 * h64, c->stream));
    const double bnorm = sqrt(bb);
    int status_conv = 0;
    double rr = 0.0;
    int iters = 0, updates = 0;

    if (bb > 0.0) {
        if (sy.even_odd) {
            // bhat_e = b_e + kappa D_eo A_oo^-1 b_o
            CK(launch_clover_apply(COLA_F64, c->g, c->clovI64, B + h64, c->tmp64, c->stream));
            c->launches++;
            ST(dslash(c, COLA_F64, 0, 0, c->tmp64, rhs, B, 0, kappa, 0, nullptr, 0));
            flops += (504.0 + 1320.0 + 48.0) * (double)c->Vh;
        }
        // CGLS; with `mixed` the inner vectors are fp32 and the fp64 residual is recomputed at reliable
        // updates that keep the search direction.  The stop / reliable-update decision is taken on
        // the device (r_update's last block raises ctl->flag); every kernel of the iteration is a no-op while the
        // flag is up, so the host queues half an iteration ahead and reads the status with a lag instead of
        // draining the stream once per iteration.
        const double target2 = (sp->tol * bnorm) * (sp->tol * bnorm);
        const double delta2 = sp->mixed ? delta * delta : 0.0;
        const cola_prec P = sp->mixed ? COLA_F32 : COLA_F64;
        char *xi = sp->mixed ? x32 : xsol, *ri = sp->mixed ? r32 : r, *pi = sp->mixed ? p32 : p, *qi = sp->mixed ? qs32 : qs;
        const size_t nvi = sp->mixed ? nv32 : nv64;
        const int nh = sy.even_odd ? 1 : 2;
        const bool deflate = c->defl_vecs && c->defl_n > 0 && sy.even_odd;
        if (deflate) {
            // x0_e = sum_i u_i <u_i, S^+ bhat_e> / lambda_i  (eigenpairs of S^+ S), r0 = bhat_e - S x0_e
            ST(apply_K(c, sy, COLA_F64, 1, rhs, qs, nullptr));
            flops += flops_K;
            for (int i = 0; i < c->defl_n; i++) {
                const char *u = c->defl_vecs + (size_t)i * h64;
                CK(launch_eig_cdot(u, qs, c->Vh, c->red, &ctl->counter[2], &ctl->aux[0], c->stream));
                CK(launch_eig_caxpy(xsol, u, c->Vh, &ctl->aux[0], 1.0 / c->defl_evals[i], c->stream));
                c->launches += 2;
            }
            ST(apply_K(c, sy, COLA_F64, 0, xsol, qs, nullptr));
            flops += flops_K;
        }
        if (sp->mixed) {
            CK(cudaMemsetAsync(x32, 0, nv32, c->stream));
            ST(axpby64(c, sy, r, 1.0, rhs, deflate ? -1.0 : 0.0, deflate ? qs : nullptr, r32));   // r64 = rhs [- S x0], r32 = float(r64)
        } else if (deflate) {
            ST(axpby64(c, sy, r, 1.0, rhs, -1.0, qs, nullptr));
        } else {
            CK(cudaMemcpyAsync(r, rhs, nv64, cudaMemcpyDeviceToDevice, c->stream));
        }
        ST(norm2(c, COLA_F64, r, sy.n_sites, &ctl->rr));
        ST(read_scalar(c, &ctl->rr, &rr));
        status_conv = rr <= target2;
        if (!status_conv) {
            ST(set_decision_state(c, rr, target2, delta2, 0));
            ST(apply_K(c, sy, P, 1, ri, qi, &ctl->gam[0]));             // s0 = K^+ r0, gamma_0
            CK(cudaMemcpyAsync(pi, qi, nvi, cudaMemcpyDeviceToDevice, c->stream));
            flops += flops_K;
            c->h_status[0].iters = c->h_status[1].iters = 0;
            ST(first_half(c, sy, P, 0, ri, pi, qi));
            for (int k = 0;; k++) {
                const int more = (k + 1 < sp->max_iter);
                ST(second_half(c, sy, P, k, 1, xi, ri, pi, qi));        // speculative: skipped if iteration k raises the flag
                if (more) ST(first_half(c, sy, P, k + 1, ri, pi, qi));
                HostStatus hs;
                ST(wait_status(c, k, &hs));
                const HostStatus *st = &hs;
                rr = st->rr;
                iters = k + 1;
                if (c->hist && k < c->hist_len) c->hist[k] = sqrt(rr) / bnorm;   // |r_{k+1}| / |b| of the recurrence
                if (!(rr <= DBL_MAX)) {   // NaN/Inf in the source or the links: no test below would ever fire
                    CK(cudaStreamSynchronize(c->stream));
                    return fail(c, COLA_EINVAL, "cola_cg_solve: the residual is not a number (NaN or Inf in the source or the gauge field)");
                }
                flops += flops_K;
                if (!st->flag) {
                    flops += flops_K;
                    if (!more) break;
                    continue;
                }
                // iteration k converged (inner residual) or asks for a reliable update; x has not received alpha_k p_k yet
                CK(launch_xp_update(P, xi, pi, qi, ctl, k & 1, 1, 0, nullptr, sy.n_sites, c->stream));
                c->launches++;
                if (!sp->mixed) { status_conv = 1; break; }
                for (int h = 0; h < nh; h++) {
                    CK(launch_accumulate(xsol + h * h64, x32 + h * h32, c->Vh, c->stream));   // x64 += x32, x32 = 0
                    c->launches++;
                }
                ST(apply_K(c, sy, COLA_F64, 0, xsol, qs, nullptr));
                flops += flops_K;
                ST(axpby64(c, sy, r, 1.0, rhs, -1.0, qs, r32));          // r64 = rhs - K x64, r32 = float(r64)
                ST(norm2(c, COLA_F64, r, sy.n_sites, &ctl->rr));
                ST(read_scalar(c, &ctl->rr, &rr));
                if (c->upd_iters && updates < c->upd_len) c->upd_iters[updates] = k + 1;
                updates++;
                if (!(rr <= DBL_MAX)) return fail(c, COLA_EINVAL, "cola_cg_solve: the fp64 residual is not a number (NaN or Inf in the gauge field)");
                if (rr <= target2) { status_conv = 1; break; }
                if (!more) break;
                ST(set_decision_state(c, rr, target2, delta2, k + 1)); // rmax = |r64|, flag down
                ST(second_half(c, sy, P, k, 0, xi, ri, pi, qi));        // same search direction: p = s + beta p
                flops += flops_K;
                ST(first_half(c, sy, P, k + 1, ri, pi, qi));
            }
            if (!status_conv && sp->mixed) {   // max_iter: fold the fp32 part into the fp64 iterate
                for (int h = 0; h < nh; h++) {
                    CK(launch_accumulate(xsol + h * h64, x32 + h * h32, c->Vh, c->stream));
                    c->launches++;
                }
            }
        }
        if (sy.even_odd) {
            // x_o = A_oo^-1 (b_o + kappa D_oe x_e)
            ST(dslash(c, COLA_F64, 1, 0, X, X + h64, B + h64, 0, kappa, 1, nullptr, 0));
            flops += (1320.0 + 48.0 + 504.0) * (double)c->Vh;
        }
    } else {
        status_conv = 1;
    }
    info->iterated_residual = bb > 0 ? sqrt(rr) / bnorm : 0.0;
    // true residual |b - M x| / |b| on the full lattice (fp64); r/qs are free now but may be half-sized: use rhs..: recompute into scratch tail
    {
        char *t = (sy.even_odd ? rhs : r);          // rhs (1 half) + r (1 half) are contiguous when even_odd; r is full-sized otherwise
        ST(fmatrix(c, COLA_F64, 0, X, t, nullptr));
        flops += 1872.0 * (double)c->V;
        double tr = 0.0;
        for (int h = 0; h < 2; h++) {
            CK(launch_axpby64(nullptr, 1.0, B + h * h64, -1.0, t + h * h64, nullptr, c->Vh, &c->red, &c->ctl->counter[3], &ctl->aux[h], c->stream));
            c->launches++;
        }
        double a0, a1;
        ST(read_scalar(c, &ctl->aux[0], &a0));
        ST(read_scalar(c, &ctl->aux[1], &a1));
        tr = a0 + a1;
        info->true_residual = bb > 0 ? sqrt(tr) / bnorm : 0.0;
    }
    CK(launch_spinor_unpack(COLA_F64, c->g, X, x_canon_dev, c->stream));
    c->launches++;
    CK(cudaEventRecord(c->ev1, c->stream));
    CK(cudaEventSynchronize(c->ev1));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, c->ev0, c->ev1));
    info->seconds = ms * 1e-3;
    info->iters = iters;
    info->reliable_updates = updates;
    info->op_flops = flops;
    if (!status_conv) return fail(c, COLA_ENOCONV, "cola_cg_solve: max_iter reached before |r| <= tol*|b|");
    return COLA_OK;
}

// ------------------------------------------------------------------------------------------------
// BiCGStab on the Schur complement ("solvers for linear systems"), van der Vorst's order as in
// oracle_bicgstab, x0 = 0, rhat = r0.  One pass = S p and S s (4 fused dslash launches) + 5 BLAS launches:
//   v = S p;  rv = <rhat, v>;  s = r - alpha v;  t = S s (|t|^2 fused);  ts = <t, s>;
//   x += alpha p + omega s, r = s - omega t, |r|^2, rho' = <rhat, r>, beta, decision;   p = r + beta (p - omega v)
// alpha, omega, beta are formed on the device (CtlB); the host queues half a pass ahead and polls the status the x/r
// update publishes, exactly as in the CGNR driver.  With `mixed` the pass runs in fp32 (or on the 16-bit fields) and
// reliable updates recompute the fp64 residual, keep p and v and re-form rho' with the replaced residual (SURVEY O8's
// schedule applied to BiCGStab).
// ------------------------------------------------------------------------------------------------
namespace {

cola_status bicg_first_half(cola_ctx *c, const System &sy, cola_prec P, int k, char *xi, char *ri, char *rhat, char *pi, char *vi, char *si, char *ti)
{
    CtlB *cb = c->ctlb;
    ST(apply_K(c, sy, P, 0, pi, vi, nullptr, &cb->flag));
    CK(launch_bicg_dot(P, rhat, vi, cb, 0, &cb->flag, sy.n_sites, c->red, c->stream));
    CK(launch_bicg_s_update(P, si, ri, vi, cb, &cb->flag, sy.n_sites, c->stream));
    ST(apply_K(c, sy, P, 0, si, ti, &cb->tt, &cb->flag, cb->ts));   // t = S s with |t|^2 and <t, s> from the same kernel (s and t are in its registers)
    CK(launch_bicg_xr_update(P, xi, ri, pi, si, ti, rhat, cb, k + 1, &cb->flag, c->d_status + (k & 1), sy.n_sites, c->red, c->stream));
    c->launches += 3;
    return COLA_OK;
}

cola_status bicg_set_decision_state(cola_ctx *c, double rmax2, double target2, double delta2, int iters)
{
    struct { double rmax2, target2, delta2; int flag, iters; } st = {rmax2, target2, delta2, 0, iters};
    static_assert(offsetof(CtlB, iters) - offsetof(CtlB, rmax2) == 28, "decision block layout");
    CK(cudaMemcpyAsync(&c->ctlb->rmax2, &st, sizeof(st), cudaMemcpyHostToDevice, c->stream));
    return COLA_OK;
}

}  // namespace

static cola_status solve_bicgstab_impl(cola_ctx *c, const cola_solve_params *sp, const void *b_canon_dev, void *x_canon_dev, cola_solve_info *info)
{
    ST(need_ready(c, "cola_cg_solve"));
    if (!sp || !b_canon_dev || !x_canon_dev || !info) return fail(c, COLA_EINVAL, "cola_cg_solve: NULL argument");
    if (!(sp->tol > 0) || sp->max_iter < 1) return fail(c, COLA_EINVAL, "cola_cg_solve: tol must be > 0 and max_iter >= 1");
    CK(cudaSetDevice(c->p.device));
    memset(info, 0, sizeof(*info));
    if (sp->mixed < 0 || sp->mixed > 3) return fail(c, COLA_EINVAL, "cola_cg_solve: mixed must be 0, 1, 2 or 3");
    if (!sp->even_odd) return fail(c, COLA_EINVAL, "cola_cg_solve: BiCGStab is offered on the Schur system only (even_odd = 1)");
    if (sp->mixed == 2) ST(check_prec(c, COLA_F32_H16, 0, 0));
    if (sp->mixed == 3) ST(check_prec(c, COLA_F32_R8, 0, 0));
    c->inner_prec = sp->mixed == 2 ? COLA_F32_H16 : (sp->mixed == 3 ? COLA_F32_R8 : COLA_F32);
    const double delta = sp->delta > 0 ? sp->delta : 0.1;
    const double kappa = c->p.kappa;
    const size_t h64 = half_bytes(c, COLA_F64), h32 = half_bytes(c, COLA_F32);
    System sy;
    sy.even_odd = 1;
    sy.n_sites = c->Vh;
    const double flops_K = 3696.0 * (double)c->Vh;
    double flops = 0.0;

    // scratch (9 fp64 half slots, as the even-odd CGNR): B 2, X 2, rhs 1, r 1, qs 1, F 2.  During the passes X's odd half
    // is free (x_o is reconstructed at the end) and, in the mixed mode, qs is only live inside a reliable update, when the
    // temporaries s and t of the pass are dead.
    char *sc = c->scratch;
    char *B = sc; sc += 2 * h64;
    char *X = sc; sc += 2 * h64;
    char *rhs = sc; sc += h64;
    char *r = sc; sc += h64;
    char *qs = sc; sc += h64;
    char *F = sc; sc += 2 * h64;
    if ((size_t)(sc - c->scratch) > c->scratch_bytes) return fail(c, COLA_ENOMEM, "cola_cg_solve: internal scratch too small");
    char *xsol = X;
    char *xi, *ri, *rhat, *pi, *vi, *si, *ti;
    if (sp->mixed) {
        xi = F; ri = F + h32; rhat = F + 2 * h32; pi = F + 3 * h32;
        vi = X + h64;
        si = qs; ti = qs + h32;
    } else {
        xi = xsol; ri = r; rhat = rhs; pi = F; si = F + h64; vi = qs; ti = X + h64;
    }
    const cola_prec P = sp->mixed ? COLA_F32 : COLA_F64;
    const size_t nvi = sp->mixed ? h32 : h64;

    Ctl *ctl = c->ctl;
    CtlB *cb = c->ctlb;
    CK(cudaEventRecord(c->ev0, c->stream));
    CK(launch_spinor_pack(COLA_F64, c->g, b_canon_dev, B, c->stream));
    c->launches++;
    double bb = 0.0;
    ST(norm2(c, COLA_F64, B, c->V, &ctl->aux[2]));
    ST(read_scalar(c, &ctl->aux[2], &bb));
    if (!(bb <= DBL_MAX)) return fail(c, COLA_EINVAL, "cola_cg_solve: the source contains NaN or Inf");
    CK(cudaMemsetAsync(X, 0, 2 * h64, c->stream));
    const double bnorm = sqrt(bb);
    int status_conv = 0;
    double rr = 0.0;
    int iters = 0, updates = 0;

    if (bb > 0.0) {
        CK(launch_clover_apply(COLA_F64, c->g, c->clovI64, B + h64, c->tmp64, c->stream));
        c->launches++;
        ST(dslash(c, COLA_F64, 0, 0, c->tmp64, rhs, B, 0, kappa, 0, nullptr, 0));     // bhat_e = b_e + kappa D_eo A_oo^-1 b_o
        flops += (504.0 + 1320.0 + 48.0) * (double)c->Vh;
        const double target2 = (sp->tol * bnorm) * (sp->tol * bnorm);
        const double delta2 = sp->mixed ? delta * delta : 0.0;
        if (sp->mixed) {
            CK(cudaMemsetAsync(xi, 0, h32, c->stream));
            ST(axpby64(c, sy, r, 1.0, rhs, 0.0, nullptr, ri));                       // r64 = rhs, r32 = float(r64)
            CK(cudaMemcpyAsync(rhat, ri, h32, cudaMemcpyDeviceToDevice, c->stream));
        } else {
            CK(cudaMemcpyAsync(ri, rhs, h64, cudaMemcpyDeviceToDevice, c->stream));
        }
        CK(cudaMemcpyAsync(pi, ri, nvi, cudaMemcpyDeviceToDevice, c->stream));
        ST(norm2(c, COLA_F64, sp->mixed ? r : ri, sy.n_sites, &ctl->rr));
        ST(read_scalar(c, &ctl->rr, &rr));
        status_conv = rr <= target2;
        if (!status_conv) {
            CtlB init;
            memset(&init, 0, sizeof(init));
            init.rv[0] = init.ts[0] = init.tt = 1.0;    // so that the beta formed with rho_next below is a number (it is not used)
            init.rho[0] = 1.0;
            init.rmax2 = rr; init.target2 = target2; init.delta2 = delta2;
            CK(cudaMemcpyAsync(cb, &init, sizeof(init), cudaMemcpyHostToDevice, c->stream));
            CK(launch_bicg_dot(P, rhat, ri, cb, 2, nullptr, sy.n_sites, c->red, c->stream));   // rho_1 = <rhat, r_0>
            c->launches++;
            c->h_status[0].iters = c->h_status[1].iters = 0;
            ST(bicg_first_half(c, sy, P, 0, xi, ri, rhat, pi, vi, si, ti));
            for (int k = 0;; k++) {
                const int more = (k + 1 < sp->max_iter);
                CK(launch_bicg_p_update(P, pi, ri, vi, cb, &cb->flag, sy.n_sites, c->stream));      // speculative: skipped if pass k raises the flag
                c->launches++;
                if (more) ST(bicg_first_half(c, sy, P, k + 1, xi, ri, rhat, pi, vi, si, ti));
                HostStatus hs;
                ST(wait_status(c, k, &hs));
                rr = hs.rr;
                iters = k + 1;
                if (c->hist && k < c->hist_len) c->hist[k] = sqrt(rr) / bnorm;
                if (!(rr <= DBL_MAX)) {
                    CK(cudaStreamSynchronize(c->stream));
                    return fail(c, COLA_EINVAL, "cola_cg_solve: BiCGStab broke down or met NaN/Inf (<rhat, v>, <t, t> or rho vanished, or bad input)");
                }
                flops += 2 * flops_K;
                if (!hs.flag) {
                    if (!more) break;
                    continue;
                }
                if (!sp->mixed) { status_conv = 1; break; }
                CK(launch_accumulate(xsol, xi, c->Vh, c->stream));                   // x64 += x32, x32 = 0
                c->launches++;
                ST(apply_K(c, sy, COLA_F64, 0, xsol, qs, nullptr));
                flops += flops_K;
                ST(axpby64(c, sy, r, 1.0, rhs, -1.0, qs, ri));                        // r64 = rhs - S x64, r32 = float(r64)
                ST(norm2(c, COLA_F64, r, sy.n_sites, &ctl->rr));
                ST(read_scalar(c, &ctl->rr, &rr));
                if (c->upd_iters && updates < c->upd_len) c->upd_iters[updates] = k + 1;
                updates++;
                if (!(rr <= DBL_MAX)) return fail(c, COLA_EINVAL, "cola_cg_solve: the fp64 residual is not a number (NaN or Inf in the gauge field)");
                if (rr <= target2) { status_conv = 1; break; }
                if (!more) break;
                ST(bicg_set_decision_state(c, rr, target2, delta2, k + 1));            // rmax = |r64|, flag down
                CK(launch_bicg_dot(P, rhat, ri, cb, 2, nullptr, sy.n_sites, c->red, c->stream));   // rho' and beta with the replaced residual
                CK(launch_bicg_p_update(P, pi, ri, vi, cb, nullptr, sy.n_sites, c->stream));   // same p and v: p = r + beta (p - omega v)
                c->launches += 2;
                ST(bicg_first_half(c, sy, P, k + 1, xi, ri, rhat, pi, vi, si, ti));
            }
            if (!status_conv && sp->mixed) {
                CK(launch_accumulate(xsol, xi, c->Vh, c->stream));
                c->launches++;
            }
        }
        ST(dslash(c, COLA_F64, 1, 0, X, X + h64, B + h64, 0, kappa, 1, nullptr, 0));   // x_o = A_oo^-1 (b_o + kappa D_oe x_e)
        flops += (1320.0 + 48.0 + 504.0) * (double)c->Vh;
    } else {
        status_conv = 1;
    }
    info->iterated_residual = bb > 0 ? sqrt(rr) / bnorm : 0.0;
    {
        char *t = rhs;          // rhs (1 half) + r (1 half) are contiguous
        ST(fmatrix(c, COLA_F64, 0, X, t, nullptr));
        flops += 1872.0 * (double)c->V;
        for (int h = 0; h < 2; h++) {
            CK(launch_axpby64(nullptr, 1.0, B + h * h64, -1.0, t + h * h64, nullptr, c->Vh, &c->red, &c->ctl->counter[3], &ctl->aux[h], c->stream));
            c->launches++;
        }
        double a0, a1;
        ST(read_scalar(c, &ctl->aux[0], &a0));
        ST(read_scalar(c, &ctl->aux[1], &a1));
        info->true_residual = bb > 0 ? sqrt(a0 + a1) / bnorm : 0.0;
    }
    CK(launch_spinor_unpack(COLA_F64, c->g, X, x_canon_dev, c->stream));
    c->launches++;
    CK(cudaEventRecord(c->ev1, c->stream));
    CK(cudaEventSynchronize(c->ev1));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, c->ev0, c->ev1));
    info->seconds = ms * 1e-3;
    info->iters = iters;
    info->reliable_updates = updates;
    info->op_flops = flops;
    if (!status_conv) return fail(c, COLA_ENOCONV, "cola_cg_solve: max_iter reached before |r| <= tol*|b|");
    return COLA_OK;
}

// ------------------------------------------------------------------------------------------------
// Low modes of H = S^+ S by thick-restart Lanczos on a Chebyshev polynomial of H (include/cola.h).
// With A' = ((hi + lo) - 2 H) / (hi - lo) the eigenvalues of H below lo map to A' > 1 and T_p(A') grows like
// cosh(p acosh A') there, while [lo, hi] stays inside [-1, 1]: the wanted modes become the LARGEST, well separated
// eigenvalues of Op = T_p(A'), which Lanczos finds in a few restarts.  Each step orthogonalises the new vector against the
// whole basis (classical Gram-Schmidt, twice), so the projected matrix T_ij = <v_i, Op v_j> is taken from the dots as
// they come; at a restart the basis is rotated onto the best Ritz vectors and the last Lanczos vector is kept (Wu &
// Simon's thick restart).  Eigenvalues of H are the Rayleigh quotients of the final Ritz vectors.
// ------------------------------------------------------------------------------------------------
namespace {

struct EigPlan {
    int n_ev, m, keep, p, max_restarts;
    double tol;
    size_t nvec, scal_off, total;
};

EigPlan eig_plan(const cola_ctx *c, const cola_eig_params *ep)
{
    EigPlan q;
    memset(&q, 0, sizeof(q));
    q.n_ev = ep->n_ev;
    q.m = ep->n_kr > 0 ? ep->n_kr : 2 * ep->n_ev + 8;
    if (q.m > 64) q.m = 64;
    q.keep = (q.m + q.n_ev) / 2;
    q.p = ep->cheb_order > 0 ? ep->cheb_order : 24;
    q.max_restarts = ep->max_restarts > 0 ? ep->max_restarts : 100;
    q.tol = ep->tol > 0 ? ep->tol : 1e-10;
    q.nvec = (size_t)q.m + 1 + (size_t)q.keep + 4;          // basis, rotation target, w, two Chebyshev vectors, S x
    q.scal_off = align_up(q.nvec * half_bytes(c, COLA_F64));
    q.total = q.scal_off + align_up((size_t)(2 * (q.m + 4) + q.m * q.m) * sizeof(double));
    return q;
}

}  // namespace

extern "C" size_t cola_eig_workspace_bytes(const cola_ctx *c, const cola_eig_params *ep)
{
    if (!c || !ep || ep->n_ev < 1 || ep->n_ev > 32) return 0;
    return eig_plan(c, ep).total;
}

// One run of the filtered Lanczos with a given window.  After convergence the window is verified (see the end of the
// function); if it was wrong the run is repeated with a corrected window, at most EIG_MAX_ATTEMPTS times in all.
static const int EIG_MAX_ATTEMPTS = 4;
static cola_status eig_lowest_run(cola_ctx *c, const cola_eig_params *ep, void *work_dev, size_t work_bytes, double *evals_host, double *resid_host,
                                  void *evecs_dev, cola_eig_info *info, int attempt)
{
    ST(need_ready(c, "cola_eig_lowest"));
    if (!ep || !work_dev || !evals_host || !resid_host || !info) return fail(c, COLA_EINVAL, "cola_eig_lowest: NULL argument");
    if (ep->n_ev < 1 || ep->n_ev > 32) return fail(c, COLA_EINVAL, "cola_eig_lowest: n_ev must be 1..32");
    const EigPlan q = eig_plan(c, ep);
    if (q.m < q.n_ev + 2) return fail(c, COLA_EINVAL, "cola_eig_lowest: n_kr must be at least n_ev + 2 (and at most 64)");
    if ((size_t)q.m > 12 * c->Vh) return fail(c, COLA_EINVAL, "cola_eig_lowest: the Krylov space is larger than the lattice's vector space");
    if (((uintptr_t)work_dev & 255) || work_bytes < q.total) return fail(c, COLA_ENOMEM, "cola_eig_lowest: workspace misaligned or smaller than cola_eig_workspace_bytes()");
    CK(cudaSetDevice(c->p.device));
    memset(info, 0, sizeof(*info));
    const size_t h64 = half_bytes(c, COLA_F64), Vh = c->Vh;
    const int m = q.m, n_ev = q.n_ev, keep = q.keep, p = q.p;
    char *base = (char *)work_dev;
    auto vec = [&](size_t i) { return base + i * h64; };
    char *V = vec(0);                              // m + 1 basis vectors
    char *R = vec((size_t)m + 1);                  // keep rotated vectors
    char *W = vec((size_t)m + 1 + keep), *T0 = W + h64, *T1 = T0 + h64, *U = T1 + h64;
    double *coef = (double *)(base + q.scal_off);  // 2 (m + 4) doubles: dots
    double *Ydev = coef + 2 * (m + 4);
    double *hcoef = new double[2 * (m + 4)];
    double *Tm = new double[(size_t)m * m], *Tw = new double[(size_t)m * m], *th = new double[m], *Y = new double[(size_t)m * m], *Ysel = new double[(size_t)m * m];
    auto cleanup = [&]() { delete[] hcoef; delete[] Tm; delete[] Tw; delete[] th; delete[] Y; delete[] Ysel; };
    int ops = 0;
#define EK(call)                                                                                          \
    do {                                                                                                  \
        cudaError_t e__ = (call);                                                                         \
        if (e__ != cudaSuccess) { cleanup(); return fail(c, COLA_ECUDA, "%s: %s", #call, cudaGetErrorString(e__)); } \
    } while (0)
#define ES(call)                                      \
    do {                                              \
        cola_status s__ = (call);                     \
        if (s__ != COLA_OK) { cleanup(); return s__; } \
    } while (0)
    auto H = [&](const char *x, char *out) -> cola_status {     // out = S^+ S x
        ST(schur(c, COLA_F64, 0, x, U, nullptr));
        ST(schur(c, COLA_F64, 1, U, out, nullptr));
        ops++;
        return COLA_OK;
    };
    auto fetch = [&](int n2) -> cola_status {                   // coef[0 .. n2) -> hcoef
        CK(cudaMemcpyAsync(hcoef, coef, sizeof(double) * n2, cudaMemcpyDeviceToHost, c->stream));
        CK(cudaStreamSynchronize(c->stream));
        return COLA_OK;
    };
    EK(cudaEventRecord(c->ev0, c->stream));
    // start vector, normalised
    EK(launch_eig_start(W, Vh, 0x2302008500ull + ep->seed, c->stream));
    EK(launch_eig_cdot(W, W, Vh, c->red, &c->ctl->counter[2], coef, c->stream));
    EK(launch_eig_normalise(V, W, Vh, coef, c->stream));
    // filter window
    double hi = ep->cheb_hi, lo = ep->cheb_lo;
    if (!(hi > 0)) {   // power iteration on H from the start vector: a lower bound of lambda_max, widened by 15 %
        EK(cudaMemcpyAsync(T0, V, h64, cudaMemcpyDeviceToDevice, c->stream));
        double lam = 0.0;
        for (int it = 0; it < 20; it++) {
            ES(H(T0, T1));
            EK(launch_eig_cdot(T1, T1, Vh, c->red, &c->ctl->counter[2], coef, c->stream));
            EK(launch_eig_normalise(T0, T1, Vh, coef, c->stream));
            ES(fetch(2));
            lam = sqrt(hcoef[0]);     // |H x| with |x| = 1
        }
        hi = 1.15 * lam;
    }
    if (!(lo > 0) || lo >= hi) lo = hi / 10.0;
    info->cheb_lo = lo;
    info->cheb_hi = hi;
    const double ca = -2.0 / (hi - lo), cb = (hi + lo) / (hi - lo);   // A' = ca H + cb
    auto Op = [&](const char *x, char *out) -> cola_status {   // out = T_p(A') x
        ST(H(x, out));
        // t1 = ca H x + cb x
        char *t1 = out;
        CK(launch_eig_lincomb(t1, ca, t1, cb, x, 0.0, nullptr, Vh, c->stream));
        if (p == 1) return COLA_OK;
        // three-term recurrence with t0 = x: t_{k+1} = 2 A' t_k - t_{k-1}; buffers rotate between out, T0, T1
        char *tkm1 = T0, *tk = T1, *tn = out;
        CK(cudaMemcpyAsync(tkm1, x, h64, cudaMemcpyDeviceToDevice, c->stream));
        CK(cudaMemcpyAsync(tk, t1, h64, cudaMemcpyDeviceToDevice, c->stream));
        for (int k = 1; k < p; k++) {
            ST(H(tk, tn));
            CK(launch_eig_lincomb(tn, 2.0 * ca, tn, 2.0 * cb, tk, -1.0, tkm1, Vh, c->stream));
            char *old = tkm1;
            tkm1 = tk; tk = tn; tn = old;
        }
        if (tk != out) CK(cudaMemcpyAsync(out, tk, h64, cudaMemcpyDeviceToDevice, c->stream));
        return COLA_OK;
    };

    memset(Tm, 0, sizeof(double) * m * m);
    int k0 = 0, restarts = 0, converged = 0, raise_lo = 0;
    double beta_m = 0.0;
    for (;; restarts++) {
        for (int j = k0; j < m; j++) {
            ES(Op(vec(j), W));
            // classical Gram-Schmidt against v_0 .. v_j, twice; the first-pass dots are column j of T
            for (int pass = 0; pass < 2; pass++) {
                for (int i = 0; i <= j; i++) EK(launch_eig_cdot(vec(i), W, Vh, c->red, &c->ctl->counter[2], coef + 2 * i, c->stream));
                for (int i = 0; i <= j; i++) EK(launch_eig_caxpy(W, vec(i), Vh, coef + 2 * i, -1.0, c->stream));
                ES(fetch(2 * (j + 1)));
                for (int i = 0; i <= j; i++) {
                    if (pass == 0) Tm[i * m + j] = Tm[j * m + i] = hcoef[2 * i];
                    else Tm[i * m + j] = (Tm[j * m + i] += hcoef[2 * i]);
                }
            }
            EK(launch_eig_cdot(W, W, Vh, c->red, &c->ctl->counter[2], coef, c->stream));
            EK(launch_eig_normalise(vec(j + 1), W, Vh, coef, c->stream));
            ES(fetch(2));
            beta_m = sqrt(hcoef[0]);
            if (!(beta_m <= DBL_MAX)) { cleanup(); return fail(c, COLA_EINVAL, "cola_eig_lowest: the Lanczos vector is not a number (NaN or Inf in the gauge field?)"); }
            c->launches += 4 * (j + 1) + 2;
        }
        memcpy(Tw, Tm, sizeof(double) * m * m);
        jacobi_eigh(m, Tw, th, Y);                                  // ascending: the wanted pairs are the LAST n_ev
        double worst = 0.0;
        for (int q2 = 0; q2 < n_ev; q2++) {
            const double est = fabs(beta_m * Y[(m - 1) * m + (m - 1 - q2)]);
            if (est > worst) worst = est;
        }
        converged = worst <= q.tol * fabs(th[m - 1]);
        if (converged || restarts + 1 >= q.max_restarts) break;
        // The n_ev-th largest Ritz value never exceeds the n_ev-th largest eigenvalue of T_p (interlacing).  If it is still
        // inside [-1, 1] after several restarts, fewer than n_ev modes are likely to lie below cheb_lo, and the run would
        // grind through max_restarts on the dense band: stop and repeat with a higher lower edge (see the end).
        if (restarts >= 4 && th[m - n_ev] <= 1.0 && lo < 0.5 * hi && attempt + 1 < EIG_MAX_ATTEMPTS) {
            raise_lo = 1;
            break;
        }
        // thick restart: keep the `keep` largest Ritz pairs and the last Lanczos vector
        for (int j = 0; j < m; j++)
            for (int q2 = 0; q2 < keep; q2++) Ysel[j * keep + q2] = Y[j * m + (m - 1 - q2)];
        EK(cudaMemcpyAsync(Ydev, Ysel, sizeof(double) * m * keep, cudaMemcpyHostToDevice, c->stream));
        EK(launch_eig_rotate(R, V, h64, m, keep, Ydev, Vh, c->stream));
        EK(cudaMemcpyAsync(V, R, (size_t)keep * h64, cudaMemcpyDeviceToDevice, c->stream));
        EK(cudaMemcpyAsync(vec(keep), vec(m), h64, cudaMemcpyDeviceToDevice, c->stream));
        EK(cudaStreamSynchronize(c->stream));                      // Ysel is reused by the host
        memset(Tm, 0, sizeof(double) * m * m);
        for (int q2 = 0; q2 < keep; q2++) {
            Tm[q2 * m + q2] = th[m - 1 - q2];
            Tm[q2 * m + keep] = Tm[keep * m + q2] = beta_m * Y[(m - 1) * m + (m - 1 - q2)];
        }
        k0 = keep;
    }
    if (raise_lo) {
        EK(cudaEventRecord(c->ev1, c->stream));
        EK(cudaEventSynchronize(c->ev1));
        float ms0 = 0.f;
        EK(cudaEventElapsedTime(&ms0, c->ev0, c->ev1));
        cleanup();
        cola_eig_params e2 = *ep;
        e2.cheb_hi = hi;
        e2.cheb_lo = (3.0 * lo < 0.5 * hi) ? 3.0 * lo : 0.5 * hi;
        const int restarts0 = restarts + 1, ops0 = ops;
        const cola_status st = eig_lowest_run(c, &e2, work_dev, work_bytes, evals_host, resid_host, evecs_dev, info, attempt + 1);
        info->seconds += ms0 * 1e-3;
        info->restarts += restarts0;
        info->op_applications += ops0;
        return st;
    }
    // final Ritz vectors of the wanted pairs -> R[0 .. n_ev), Rayleigh quotients and true residuals with H
    for (int j = 0; j < m; j++)
        for (int q2 = 0; q2 < n_ev; q2++) Ysel[j * n_ev + q2] = Y[j * m + (m - 1 - q2)];
    EK(cudaMemcpyAsync(Ydev, Ysel, sizeof(double) * m * n_ev, cudaMemcpyHostToDevice, c->stream));
    EK(launch_eig_rotate(R, V, h64, m, n_ev, Ydev, Vh, c->stream));
    double lam[32], res[32];
    int order[32];
    for (int q2 = 0; q2 < n_ev; q2++) {
        char *u = R + (size_t)q2 * h64;
        EK(launch_eig_cdot(u, u, Vh, c->red, &c->ctl->counter[2], coef, c->stream));     // renormalise (rotation rounding)
        EK(launch_eig_normalise(u, u, Vh, coef, c->stream));
        ES(H(u, W));
        EK(launch_eig_cdot(u, W, Vh, c->red, &c->ctl->counter[2], coef + 2, c->stream));
        EK(launch_eig_caxpy(W, u, Vh, coef + 2, -1.0, c->stream));
        EK(launch_eig_cdot(W, W, Vh, c->red, &c->ctl->counter[2], coef + 4, c->stream));
        ES(fetch(6));
        lam[q2] = hcoef[2];
        res[q2] = sqrt(hcoef[4]);
        order[q2] = q2;
    }
    for (int a = 0; a < n_ev; a++)
        for (int b2 = a + 1; b2 < n_ev; b2++)
            if (lam[order[b2]] < lam[order[a]]) { const int t = order[a]; order[a] = order[b2]; order[b2] = t; }
    for (int a = 0; a < n_ev; a++) {
        evals_host[a] = lam[order[a]];
        resid_host[a] = res[order[a]];
        if (evecs_dev) EK(cudaMemcpyAsync((char *)evecs_dev + (size_t)a * h64, R + (size_t)order[a] * h64, h64, cudaMemcpyDeviceToDevice, c->stream));
    }
    EK(cudaEventRecord(c->ev1, c->stream));
    EK(cudaEventSynchronize(c->ev1));
    float ms = 0.f;
    EK(cudaEventElapsedTime(&ms, c->ev0, c->ev1));
    info->seconds = ms * 1e-3;
    info->restarts = restarts + 1;
    info->op_applications = ops;
    cleanup();
#undef EK
#undef ES
    if (!converged) return fail(c, COLA_ENOCONV, "cola_eig_lowest: max_restarts reached before the residual estimates met tol");
    // Was the window right?  The filter T_p maps eigenvalues of H below cheb_lo to values > 1, monotonically (smaller
    // lambda, larger value), and [cheb_lo, cheb_hi] into [-1, 1]; the run returns the n_ev LARGEST Ritz pairs of T_p.
    // Those are the n_ev smallest eigenpairs of H only if (a) at least n_ev eigenvalues lie below cheb_lo -- otherwise the
    // list is padded with modes of the oscillating band, in no particular order -- and (b) nothing lies above cheb_hi -- an
    // even-order T_p sends such modes to large positive values as well, and the power iteration behind the default cheb_hi
    // only bounds lambda_max from below.  Both failures show in the Rayleigh quotients just computed with H itself: a
    // returned lambda >= cheb_lo.  (The residuals are small either way, so they cannot tell.)
    double lam_max = evals_host[n_ev - 1];
    if (lam_max < lo) return COLA_OK;
    cola_eig_params e2 = *ep;
    e2.cheb_hi = hi;
    e2.cheb_lo = lo;
    if (lam_max > hi) e2.cheb_hi = 1.15 * lam_max;                        // (b): an eigenvalue above the window
    else e2.cheb_lo = (2.0 * lam_max < 0.5 * hi) ? 2.0 * lam_max : 0.5 * (lam_max + hi);   // (a): raise the lower edge past it
    if (!(e2.cheb_lo < e2.cheb_hi)) e2.cheb_lo = 0.5 * e2.cheb_hi;
    if (attempt + 1 >= EIG_MAX_ATTEMPTS)
        return fail(c, COLA_ENOCONV, "cola_eig_lowest: a returned eigenvalue lies at or above cheb_lo after the window was corrected repeatedly: "
                                     "the pairs are converged eigenpairs of S^+S but not certified as the lowest; pass cheb_lo / cheb_hi explicitly");
    const cola_eig_info first = *info;
    const cola_status st = eig_lowest_run(c, &e2, work_dev, work_bytes, evals_host, resid_host, evecs_dev, info, attempt + 1);
    info->seconds += first.seconds;          // account for every run
    info->restarts += first.restarts;
    info->op_applications += first.op_applications;
    return st;
}

extern "C" cola_status cola_eig_lowest(cola_ctx *c, const cola_eig_params *ep, void *work_dev, size_t work_bytes, double *evals_host, double *resid_host,
                                       void *evecs_dev, cola_eig_info *info)
{
    return eig_lowest_run(c, ep, work_dev, work_bytes, evals_host, resid_host, evecs_dev, info, 0);
}

extern "C" cola_status cola_cg_solve_deflated(cola_ctx *c, const cola_solve_params *sp, const void *b_canon_dev, void *x_canon_dev, cola_solve_info *info,
                                              const void *evecs_dev, const double *evals_host, int n_ev)
{
    if (!c) return COLA_EINVAL;
    if (!evecs_dev || !evals_host || n_ev < 1) return fail(c, COLA_EINVAL, "cola_cg_solve_deflated: NULL or empty eigenpairs");
    if (!sp || !sp->even_odd || sp->method != COLA_CGNR) return fail(c, COLA_EINVAL, "cola_cg_solve_deflated: needs even_odd = 1 and method = COLA_CGNR");
    for (int i = 0; i < n_ev; i++)
        if (!(evals_host[i] > 0)) return fail(c, COLA_EINVAL, "cola_cg_solve_deflated: eigenvalues of S^+S must be positive");
    c->defl_vecs = (const char *)evecs_dev;
    c->defl_evals = evals_host;
    c->defl_n = n_ev;
    const cola_status st = solve_impl(c, sp, b_canon_dev, x_canon_dev, info);
    c->defl_vecs = nullptr;
    c->defl_evals = nullptr;
    c->defl_n = 0;
    return st;
}

// ------------------------------------------------------------------------------------------------
// multi-right-hand-side operators and batched solver
// ------------------------------------------------------------------------------------------------
namespace {

struct CarveM {
    size_t tmp32, r64, partials, op_total;          // what the multi-rhs operators need
    size_t rhs, qs, x32, r32, p32, q32, rhat32, ctlb, total;      // + the vectors of the batched solvers
    int nsb;
};

CarveM carve_m(const cola_ctx *c, int nrhs)
{
    CarveM k;
    size_t off = 0;
    const size_t h64 = half_bytes(c, COLA_F64), h32 = half_bytes(c, COLA_F32), n = (size_t)nrhs;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
    k.tmp32 = take(n * h32);
    k.r64 = take(n * h64);
    {
        size_t nsb = (size_t)mrhs_site_blocks(c->g);
        const size_t nb32 = (size_t)blas_mrhs_blocks(c->Vh, COLA_F32), nb64 = (size_t)blas_mrhs_blocks(c->Vh, COLA_F64);
        if (nsb < nb32) nsb = nb32;
        if (nsb < nb64) nsb = nb64;
        k.nsb = (int)nsb;
        k.partials = take(n * nsb * sizeof(double));
    }
    k.op_total = off;
    k.rhs = take(n * h64);
    k.qs = take(n * h64);
    k.x32 = take(n * h32);
    k.r32 = take(n * h32);
    k.p32 = take(n * h32);
    k.q32 = take(n * h32);
    k.rhat32 = take(n * h32);
    k.ctlb = take(MRHS_MAX * (sizeof(CtlB) + sizeof(HostStatus) + sizeof(double)));
    k.total = off;
    return k;
}

MrhsList list_of(const int *v, int n)
{
    MrhsList l;
    for (int k = 0; k < MRHS_MAX; k++) l.v[k] = k < n ? v[k] : 0;
    return l;
}

cola_status need_mrhs(cola_ctx *c, const char *who, int nrhs)
{
    ST(need_ready(c, who));
    if (nrhs < 1 || nrhs > MRHS_MAX) return fail(c, COLA_EINVAL, "%s: nrhs must be 1..16", who);
    if (c->m_nrhs < nrhs) return fail(c, COLA_ENOTREADY, "%s: no multi-rhs workspace for that many right-hand sides (call cola_set_mrhs_workspace)", who);
    return COLA_OK;
}

// batched  out_p[n] = [post] ( [A] y[n] + coef * D_{p,1-p} in[n] )  for the vectors list.v[0..nrhs);  optional |out[n]|^2 -> norm_out[n]
cola_status dslash_m(cola_ctx *c, cola_prec prec, int parity, int dagger, const MrhsList &list, int nrhs, const void *in, size_t in_stride, void *out,
                     size_t out_stride, const void *y, size_t y_stride, int clov_on_y, double coef, int post_inv, double *norm_out, int norm_accumulate,
                     const int *skip)
{
    ST(check_prec(c, prec, parity, (y && clov_on_y) ? 1 : 0));
    MrhsArgs m;
    memset(&m, 0, sizeof(m));
    DslashArgs &a = m.d;
    a.g = c->g;
    a.in = in;
    a.out = out;
    a.gauge_p = gauge_of(c, prec, parity);
    a.gauge_q = gauge_of(c, prec, 1 - parity);
    a.y = y;
    a.clov_y = (y && clov_on_y) ? clovA_of(c, prec, parity) : nullptr;
    a.clov_y_g48 = (a.clov_y && r8_clover(c, prec)) ? 1 : 0;
    a.clov_post = post_inv ? clovI_of(c, prec) : nullptr;
    a.coef = coef;
    a.sgn = dagger ? +1.0 : -1.0;
    a.parity = parity;
    a.skip = skip;
    a.sweep.zb = choose_zband(c->g.Xh * c->g.Y, c->g.Z, (size_t)(prec == COLA_F64 ? 192 : 96) * (size_t)nrhs, c->l2_budget, mrhs_tile_z(c->g));
    m.nrhs = nrhs;
    m.in_stride = in_stride;
    m.out_stride = out_stride;
    m.y_stride = y_stride;
    for (int k = 0; k < MRHS_MAX; k++) m.list[k] = list.v[k];
    m.partials = norm_out ? c->m_partials : nullptr;
    if (post_inv && parity != 1) return fail(c, COLA_EINVAL, "internal: A^-1 is stored on the odd parity only");
    CK(launch_dslash_mrhs(fmt_of(c, prec), m, c->stream));
    c->launches++;
    if (norm_out) {
        CK(launch_mrhs_reduce(c->m_partials, m.nsb, nrhs, list.v, norm_out, norm_accumulate, skip, c->stream));
        c->launches++;
    }
    return COLA_OK;
}

// batched Schur: out_e[n] = S in_e[n]; tmp = nrhs odd half vectors of precision prec (stride = half_bytes)
cola_status schur_m(cola_ctx *c, cola_prec prec, int dagger, const MrhsList &list, int nrhs, const void *in, size_t in_stride, void *tmp, void *out,
                    size_t out_stride, double *norm_out, const int *skip)
{
    const double k = c->p.kappa;
    const size_t hb = half_bytes(c, prec);
    ST(dslash_m(c, prec, 1, dagger, list, nrhs, in, in_stride, tmp, hb, nullptr, 0, 0, 0.0, 1, nullptr, 0, skip));
    ST(dslash_m(c, prec, 0, dagger, list, nrhs, tmp, hb, out, out_stride, in, in_stride, 1, -k * k, 0, norm_out, 0, skip));
    return COLA_OK;
}

}  // namespace

namespace {

cola_status wait_status_m(cola_ctx *c, int k, HostStatusM *out)
{
    volatile HostStatusM *m = c->h_statusm + (k & 1);
    for (unsigned long spins = 0;; spins++) {
        if (m->iters == k + 1) break;
        if ((spins & 0xfff) == 0xfff) {
            cudaError_t e = cudaStreamQuery(c->stream);
            if (e == cudaSuccess) {
                if (m->iters == k + 1) break;
                return fail(c, COLA_ECUDA, "cola_cg_solve_mrhs: the stream drained without iteration status (internal error)");
            }
            if (e != cudaErrorNotReady) return fail(c, COLA_ECUDA, "cola_cg_solve_mrhs: %s", cudaGetErrorString(e));
        }
        cpu_relax();
    }
    __sync_synchronize();
    for (int n = 0; n < MRHS_MAX; n++) out->rr[n] = m->rr[n];
    out->trig = m->trig;
    out->flag = m->flag;
    out->iters = m->iters;
    return COLA_OK;
}

// iteration k of the batch, first half:  q = S p (|q|^2),  r -= alpha q (|r|^2), decision -> mapped host slot k & 1
cola_status first_half_m(cola_ctx *c, int k, const MrhsList &A, int na)
{
    CtlM *cm = c->ctlm;
    const size_t h32 = half_bytes(c, COLA_F32);
    const int nb = blas_mrhs_blocks(c->Vh, COLA_F32);
    ST(schur_m(c, c->inner_prec, 0, A, na, c->m_p32, h32, c->m_tmp32, c->m_q32, h32, cm->qq, &cm->flag));
    CK(launch_r_update_mrhs(COLA_F32, c->m_r32, c->m_q32, h32, cm, k & 1, A, na, &cm->flag, c->Vh, c->m_partials, c->stream));
    CK(launch_mrhs_reduce(c->m_partials, nb, na, A.v, cm->rr, 0, &cm->flag, c->stream));
    CK(launch_decide_mrhs(cm, A, na, k + 1, &cm->flag, c->d_statusm + (k & 1), c->stream));
    c->launches += 3;
    return COLA_OK;
}

// second half:  s = S^+ r (|s|^2 -> gam[next]),  x += alpha p (do_x),  p = s + beta p
cola_status second_half_m(cola_ctx *c, int k, int do_x, const MrhsList &A, int na)
{
    CtlM *cm = c->ctlm;
    const size_t h32 = half_bytes(c, COLA_F32);
    ST(schur_m(c, c->inner_prec, 1, A, na, c->m_r32, h32, c->m_tmp32, c->m_q32, h32, cm->gam[(k & 1) ^ 1], &cm->flag));
    CK(launch_xp_update_mrhs(COLA_F32, c->m_x32, c->m_p32, c->m_q32, h32, cm, k & 1, A, na, do_x, 1, &cm->flag, c->Vh, c->stream));
    c->launches++;
    return COLA_OK;
}

}  // namespace

// Batched mixed-precision even-odd CGNR: nrhs independent systems M x_n = b_n advance in lock step so that every
// pass over the links and the clover field serves all of them.  Each system keeps its own alpha, beta, residual
// history and reliable-update schedule (SURVEY O7/O8 per system): the device raises one flag when ANY active system
// converges in the inner precision or asks for a reliable update; the host then updates exactly those systems
// (fp64 true residual, search direction kept), drops the ones that have converged and re-queues the rest.
// Storage: the internal x_n lives in the caller's x_n buffer during the solve (same size) and is unpacked in place
// at the end through the context's scratch.
static cola_status solve_mrhs_impl(cola_ctx *c, const cola_solve_params *sp, int nrhs, const void *b_canon_dev, void *x_canon_dev, cola_solve_info *infos)
{
    ST(need_mrhs(c, "cola_cg_solve_mrhs", nrhs));
    if (!sp || !b_canon_dev || !x_canon_dev || !infos) return fail(c, COLA_EINVAL, "cola_cg_solve_mrhs: NULL argument");
    if (!(sp->tol > 0) || sp->max_iter < 1) return fail(c, COLA_EINVAL, "cola_cg_solve_mrhs: tol must be > 0 and max_iter >= 1");
    if (!sp->even_odd || sp->mixed < 1 || sp->mixed > 3 || (sp->method != COLA_CGNR && sp->method != COLA_BICGSTAB))
        return fail(c, COLA_EINVAL, "cola_cg_solve_mrhs: only the mixed-precision even-odd solvers are batched (even_odd = 1, mixed = 1, 2 or 3)");
    if (sp->mixed == 2) ST(check_prec(c, COLA_F32_H16, 0, 0));
    if (sp->mixed == 3) ST(check_prec(c, COLA_F32_R8, 0, 0));
    if (!c->m_solver) return fail(c, COLA_ENOTREADY, "cola_cg_solve_mrhs: the multi-rhs workspace was sized for operators only (cola_mrhs_workspace_bytes with for_solver = 1)");
    c->inner_prec = sp->mixed == 2 ? COLA_F32_H16 : (sp->mixed == 3 ? COLA_F32_R8 : COLA_F32);
    CK(cudaSetDevice(c->p.device));
    const double delta = sp->delta > 0 ? sp->delta : 0.1, kappa = c->p.kappa;
    const size_t h64 = half_bytes(c, COLA_F64), h32 = half_bytes(c, COLA_F32), f64 = 2 * h64;
    const double flops_K = 3696.0 * (double)c->Vh;
    Ctl *ctl = c->ctl;
    CtlM *cm = c->ctlm;
    char *Bt = c->scratch, *Tt = Bt + f64;      // packed source of one system; full-lattice temporary
    char *Xall = (char *)x_canon_dev;
    const char *Ball = (const char *)b_canon_dev;
    double bb[MRHS_MAX], bnorm[MRHS_MAX], target2[MRHS_MAX], rr[MRHS_MAX], flops[MRHS_MAX];
    int conv[MRHS_MAX], iters[MRHS_MAX], updates[MRHS_MAX];
    int broken[MRHS_MAX] = {0};   // BiCGStab: systems whose recurrence produced NaN / Inf (dropped from the batch)
    memset(infos, 0, sizeof(cola_solve_info) * nrhs);
    CK(cudaEventRecord(c->ev0, c->stream));

    // ---- source preparation, one system at a time (once per solve)
    for (int n = 0; n < nrhs; n++) {
        conv[n] = iters[n] = updates[n] = 0;
        flops[n] = rr[n] = target2[n] = 0.0;
        char *X = Xall + (size_t)n * f64;
        CK(launch_spinor_pack(COLA_F64, c->g, Ball + (size_t)n * f64, Bt, c->stream));
        c->launches++;
        ST(norm2(c, COLA_F64, Bt, c->V, &ctl->aux[2]));
        ST(read_scalar(c, &ctl->aux[2], &bb[n]));
        if (!(bb[n] <= DBL_MAX)) return fail(c, COLA_EINVAL, "cola_cg_solve_mrhs: a source contains NaN or Inf");
        bnorm[n] = sqrt(bb[n]);
        CK(cudaMemsetAsync(X, 0, f64, c->stream));
        CK(cudaMemsetAsync(c->m_x32 + (size_t)n * h32, 0, h32, c->stream));
        if (!(bb[n] > 0.0)) { conv[n] = 1; continue; }
        char *rhs = c->m_rhs + (size_t)n * h64, *r = c->m_r64 + (size_t)n * h64;
        CK(launch_clover_apply(COLA_F64, c->g, c->clovI64, Bt + h64, c->tmp64, c->stream));
        c->launches++;
        ST(dslash(c, COLA_F64, 0, 0, c->tmp64, rhs, Bt, 0, kappa, 0, nullptr, 0));                       // bhat_e = b_e + kappa D_eo A_oo^-1 b_o
        flops[n] += (504.0 + 1320.0 + 48.0) * (double)c->Vh;
        CK(launch_axpby64(r, 1.0, rhs, 0.0, nullptr, c->m_r32 + (size_t)n * h32, c->Vh, &c->red, &ctl->counter[3], &cm->rr[n], c->stream));
        c->launches++;
    }
    CK(cudaMemcpyAsync(c->h_pinned, cm->rr, sizeof(double) * MRHS_MAX, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    int A[MRHS_MAX], na = 0;
    for (int n = 0; n < nrhs; n++) {
        if (conv[n]) continue;
        rr[n] = c->h_pinned[n];
        target2[n] = (sp->tol * bnorm[n]) * (sp->tol * bnorm[n]);
        if (rr[n] <= target2[n]) conv[n] = 1;
        else A[na++] = n;
    }

    if (na > 0 && sp->method == COLA_BICGSTAB) {
        // Batched BiCGStab (SURVEY 8(f) NEXT-4 on NEXT-1's kernels): the systems advance pass by pass in lock step, the two
        // applications of S per pass are multi-rhs launches over the active systems, everything else is the single-system
        // BiCGStab's own kernels and scalars (one CtlB per system), so each system follows its sequential recurrence (the
        // fused |t|^2 is summed in the multi-rhs kernels' order).  No speculative queueing: one stream synchronisation per
        // pass reads every system's |r|^2 and flag.  s and t of system n live in its fp64 slot of m_qs (K x64 of the reliable
        // update, dead during a pass), v in m_q32.
        if (!c->h_statb) CK(cudaHostAlloc(reinterpret_cast<void **>(&c->h_statb), MRHS_MAX * sizeof(HostStatus), cudaHostAllocDefault));
        const double delta2 = delta * delta;
        const cola_prec P = COLA_F32;
        const size_t nv = c->Vh;
        auto v32 = [&](char *base, int n) { return base + (size_t)n * h32; };
        auto s32 = [&](int n) { return c->m_qs + (size_t)n * h64; };
        auto t32 = [&](int n) { return c->m_qs + (size_t)n * h64 + h32; };
        for (int j = 0; j < na; j++) {
            const int n = A[j];
            CtlB init;
            memset(&init, 0, sizeof(init));
            init.rv[0] = init.ts[0] = init.tt = 1.0;
            init.rho[0] = 1.0;
            init.rmax2 = rr[n]; init.target2 = target2[n]; init.delta2 = delta2;
            CK(cudaMemcpyAsync(&c->m_ctlb[n], &init, sizeof(init), cudaMemcpyHostToDevice, c->stream));
            CK(cudaMemcpyAsync(v32(c->m_rhat32, n), v32(c->m_r32, n), h32, cudaMemcpyDeviceToDevice, c->stream));
            CK(cudaMemcpyAsync(v32(c->m_p32, n), v32(c->m_r32, n), h32, cudaMemcpyDeviceToDevice, c->stream));
            CK(launch_bicg_dot(P, v32(c->m_rhat32, n), v32(c->m_r32, n), &c->m_ctlb[n], 2, nullptr, nv, c->red, c->stream));   // rho_1 = <rhat, r_0>
            c->launches++;
        }
        CK(cudaStreamSynchronize(c->stream));   // `init` is a stack object of this loop
        for (int k = 0;; k++) {
            const int more = (k + 1 < sp->max_iter);
            const MrhsList L = list_of(A, na);
            ST(schur_m(c, c->inner_prec, 0, L, na, c->m_p32, h32, c->m_tmp32, c->m_q32, h32, nullptr, nullptr));             // v = S p
            for (int j = 0; j < na; j++) {
                const int n = A[j];
                CK(launch_bicg_dot(P, v32(c->m_rhat32, n), v32(c->m_q32, n), &c->m_ctlb[n], 0, nullptr, nv, c->red, c->stream));
                CK(launch_bicg_s_update(P, s32(n), v32(c->m_r32, n), v32(c->m_q32, n), &c->m_ctlb[n], nullptr, nv, c->stream));
            }
            ST(schur_m(c, c->inner_prec, 0, L, na, c->m_qs, h64, c->m_tmp32, c->m_qs + h32, h64, c->m_tt, nullptr));          // t = S s, |t|^2
            for (int j = 0; j < na; j++) {
                const int n = A[j];
                CK(cudaMemcpyAsync(&c->m_ctlb[n].tt, &c->m_tt[n], sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
                CK(launch_bicg_dot(P, t32(n), s32(n), &c->m_ctlb[n], 1, nullptr, nv, c->red, c->stream));
                CK(launch_bicg_xr_update(P, v32(c->m_x32, n), v32(c->m_r32, n), v32(c->m_p32, n), s32(n), t32(n), v32(c->m_rhat32, n), &c->m_ctlb[n], k + 1,
                                         nullptr, c->m_statb + n, nv, c->red, c->stream));
            }
            c->launches += 4 * (unsigned long long)na;
            CK(cudaMemcpyAsync(c->h_statb, c->m_statb, MRHS_MAX * sizeof(HostStatus), cudaMemcpyDeviceToHost, c->stream));
            CK(cudaStreamSynchronize(c->stream));
            int S[MRHS_MAX], ns = 0;
            for (int j = 0; j < na; j++) {
                const int n = A[j];
                rr[n] = c->h_statb[n].rr;
                iters[n] = k + 1;
                flops[n] += 2 * flops_K;
                if (!(rr[n] <= DBL_MAX)) {   // this system broke down: it leaves the batch with its last fp64 iterate, the others go on
                    broken[n] = 1;
                    continue;
                }
                if (c->h_statb[n].flag) S[ns++] = n;
            }
            if (ns > 0) {   // reliable updates of the systems that asked for one (or converged in the inner precision)
                for (int j = 0; j < ns; j++) {
                    CK(launch_accumulate(Xall + (size_t)S[j] * f64, v32(c->m_x32, S[j]), c->Vh, c->stream));   // x64 += x32, x32 = 0
                    c->launches++;
                }
                const MrhsList LS = list_of(S, ns);
                ST(schur_m(c, COLA_F64, 0, LS, ns, Xall, f64, c->m_r64, c->m_qs, h64, nullptr, nullptr));      // K x64 into the (dead) s / t slot
                for (int j = 0; j < ns; j++) {
                    const size_t n = (size_t)S[j];
                    CK(launch_axpby64(c->m_r64 + n * h64, 1.0, c->m_rhs + n * h64, -1.0, c->m_qs + n * h64, c->m_r32 + n * h32, c->Vh, &c->red,
                                      &ctl->counter[3], &c->m_tt[n], c->stream));                              // r64 = rhs - S x64, r32 = float(r64)
                    c->launches++;
                }
                CK(cudaMemcpyAsync(c->h_pinned, c->m_tt, sizeof(double) * MRHS_MAX, cudaMemcpyDeviceToHost, c->stream));
                CK(cudaStreamSynchronize(c->stream));
                struct { double rmax2, target2, delta2; int flag, iters; } st[MRHS_MAX];
                static_assert(offsetof(CtlB, iters) - offsetof(CtlB, rmax2) == 28, "decision block layout");
                for (int j = 0; j < ns; j++) {
                    const int n = S[j];
                    rr[n] = c->h_pinned[n];
                    updates[n]++;
                    flops[n] += flops_K;
                    if (!(rr[n] <= DBL_MAX)) return fail(c, COLA_EINVAL, "cola_cg_solve_mrhs: the fp64 residual is not a number (NaN or Inf in the gauge field)");
                    if (rr[n] <= target2[n]) { conv[n] = 1; continue; }
                    if (!more) continue;
                    st[j].rmax2 = rr[n]; st[j].target2 = target2[n]; st[j].delta2 = delta2; st[j].flag = 0; st[j].iters = k + 1;
                    CK(cudaMemcpyAsync(&c->m_ctlb[n].rmax2, &st[j], sizeof(st[j]), cudaMemcpyHostToDevice, c->stream));
                    CK(launch_bicg_dot(P, v32(c->m_rhat32, n), v32(c->m_r32, n), &c->m_ctlb[n], 2, nullptr, nv, c->red, c->stream));   // rho' and beta with the replaced residual
                    c->launches++;
                }
                CK(cudaStreamSynchronize(c->stream));   // `st` is a stack object of this block
            }
            int na2 = 0;
            for (int j = 0; j < na; j++)
                if (!conv[A[j]] && !broken[A[j]]) A[na2++] = A[j];
            na = na2;
            if (na == 0 || !more) break;
            for (int j = 0; j < na; j++) {   // p = r + beta (p - omega v)
                const int n = A[j];
                CK(launch_bicg_p_update(P, v32(c->m_p32, n), v32(c->m_r32, n), v32(c->m_q32, n), &c->m_ctlb[n], nullptr, nv, c->stream));
                c->launches++;
            }
        }
        for (int j = 0; j < na; j++) {   // max_iter: fold the fp32 parts into the fp64 iterates
            CK(launch_accumulate(Xall + (size_t)A[j] * f64, c->m_x32 + (size_t)A[j] * h32, c->Vh, c->stream));
            c->launches++;
        }
    } else if (na > 0) {
        CtlM st;
        memset(&st, 0, sizeof(st));
        for (int n = 0; n < nrhs; n++) { st.rmax2[n] = rr[n]; st.target2[n] = target2[n]; }
        st.delta2 = delta * delta;
        CK(cudaMemcpyAsync(cm, &st, sizeof(st), cudaMemcpyHostToDevice, c->stream));
        MrhsList L = list_of(A, na);
        ST(schur_m(c, c->inner_prec, 1, L, na, c->m_r32, h32, c->m_tmp32, c->m_q32, h32, cm->gam[0], nullptr));    // s0 = S^+ r0, gamma_0
        CK(cudaMemcpyAsync(c->m_p32, c->m_q32, (size_t)nrhs * h32, cudaMemcpyDeviceToDevice, c->stream));
        for (int j = 0; j < na; j++) flops[A[j]] += flops_K;
        c->h_statusm[0].iters = c->h_statusm[1].iters = 0;
        ST(first_half_m(c, 0, L, na));
        for (int k = 0;; k++) {
            const int more = (k + 1 < sp->max_iter);
            ST(second_half_m(c, k, 1, L, na));                          // speculative: skipped if iteration k raises the flag
            if (more) ST(first_half_m(c, k + 1, L, na));
            HostStatusM hs;
            ST(wait_status_m(c, k, &hs));
            for (int j = 0; j < na; j++) { rr[A[j]] = hs.rr[A[j]]; iters[A[j]] = k + 1; flops[A[j]] += flops_K; }
            for (int j = 0; j < na; j++)
                if (!(rr[A[j]] <= DBL_MAX)) {   // NaN/Inf in a source or the links: no trigger would ever fire for that system
                    CK(cudaStreamSynchronize(c->stream));
                    return fail(c, COLA_EINVAL, "cola_cg_solve_mrhs: a residual is not a number (NaN or Inf in a source or the gauge field)");
                }
            if (!hs.flag) {
                for (int j = 0; j < na; j++) flops[A[j]] += flops_K;
                if (!more) break;
                continue;
            }
            // some systems converged in fp32 or ask for a reliable update; no x has received alpha_k p_k yet
            CK(launch_xp_update_mrhs(COLA_F32, c->m_x32, c->m_p32, c->m_q32, h32, cm, k & 1, L, na, 1, 0, nullptr, c->Vh, c->stream));
            c->launches++;
            int S[MRHS_MAX], ns = 0;
            for (int j = 0; j < na; j++) if (hs.trig & (1u << A[j])) S[ns++] = A[j];
            if (ns == 0) return fail(c, COLA_ECUDA, "cola_cg_solve_mrhs: flag raised without a triggering system (internal error)");
            for (int j = 0; j < ns; j++) {
                CK(launch_accumulate(Xall + (size_t)S[j] * f64, c->m_x32 + (size_t)S[j] * h32, c->Vh, c->stream));   // x64 += x32, x32 = 0
                c->launches++;
            }
            const MrhsList LS = list_of(S, ns);
            ST(schur_m(c, COLA_F64, 0, LS, ns, Xall, f64, c->m_r64, c->m_qs, h64, nullptr, nullptr));     // r64 is dead here: it is the Schur temporary
            for (int j = 0; j < ns; j++) {
                const size_t n = (size_t)S[j];
                CK(launch_axpby64(c->m_r64 + n * h64, 1.0, c->m_rhs + n * h64, -1.0, c->m_qs + n * h64, c->m_r32 + n * h32, c->Vh, &c->red,
                                  &ctl->counter[3], &cm->rr[n], c->stream));                                  // r64 = rhs - S x64, r32 = float(r64)
                c->launches++;
            }
            CK(cudaMemcpyAsync(c->h_pinned, cm->rr, sizeof(double) * MRHS_MAX, cudaMemcpyDeviceToHost, c->stream));
            CK(cudaStreamSynchronize(c->stream));
            int na2 = 0;
            for (int j = 0; j < na; j++) {
                const int n = A[j];
                if (hs.trig & (1u << n)) {
                    rr[n] = c->h_pinned[n];
                    updates[n]++;
                    flops[n] += flops_K;
                    if (rr[n] <= target2[n]) { conv[n] = 1; continue; }
                    CK(cudaMemcpyAsync(&cm->rmax2[n], &rr[n], sizeof(double), cudaMemcpyHostToDevice, c->stream));   // rmax = |r64|
                }
                A[na2++] = n;
            }
            na = na2;
            if (na == 0 || !more) break;
            struct { int flag, iters; unsigned trig; } rearm = {0, k + 1, 0u};
            static_assert(offsetof(CtlM, trig) - offsetof(CtlM, flag) == 8, "CtlM decision block layout");
            CK(cudaMemcpyAsync(&cm->flag, &rearm, sizeof(rearm), cudaMemcpyHostToDevice, c->stream));
            L = list_of(A, na);
            ST(second_half_m(c, k, 0, L, na));                          // same search directions: p = s + beta p
            for (int j = 0; j < na; j++) flops[A[j]] += flops_K;
            ST(first_half_m(c, k + 1, L, na));
        }
        for (int j = 0; j < na; j++) {   // max_iter: fold the fp32 parts into the fp64 iterates
            CK(launch_accumulate(Xall + (size_t)A[j] * f64, c->m_x32 + (size_t)A[j] * h32, c->Vh, c->stream));
            c->launches++;
        }
    }

    // ---- reconstruction of the odd sites, fp64 true residual and unpacking, one system at a time
    int all_conv = 1;
    for (int n = 0; n < nrhs; n++) {
        char *X = Xall + (size_t)n * f64;
        double tr = 0.0;
        if (bb[n] > 0.0) {
            CK(launch_spinor_pack(COLA_F64, c->g, Ball + (size_t)n * f64, Bt, c->stream));
            c->launches++;
            ST(dslash(c, COLA_F64, 1, 0, X, X + h64, Bt + h64, 0, kappa, 1, nullptr, 0));               // x_o = A_oo^-1 (b_o + kappa D_oe x_e)
            flops[n] += (1320.0 + 48.0 + 504.0) * (double)c->Vh;
            ST(fmatrix(c, COLA_F64, 0, X, Tt, nullptr));
            flops[n] += 1872.0 * (double)c->V;
            for (int h = 0; h < 2; h++) {
                CK(launch_axpby64(nullptr, 1.0, Bt + h * h64, -1.0, Tt + h * h64, nullptr, c->Vh, &c->red, &ctl->counter[3], &ctl->aux[h], c->stream));
                c->launches++;
            }
            double a0, a1;
            ST(read_scalar(c, &ctl->aux[0], &a0));
            ST(read_scalar(c, &ctl->aux[1], &a1));
            tr = a0 + a1;
        }
        CK(launch_spinor_unpack(COLA_F64, c->g, X, Tt, c->stream));
        c->launches++;
        CK(cudaMemcpyAsync(X, Tt, f64, cudaMemcpyDeviceToDevice, c->stream));
        infos[n].iters = iters[n];
        infos[n].reliable_updates = updates[n];
        infos[n].iterated_residual = bb[n] > 0 ? sqrt(rr[n]) / bnorm[n] : 0.0;
        infos[n].true_residual = bb[n] > 0 ? sqrt(tr) / bnorm[n] : 0.0;
        infos[n].op_flops = flops[n];
        if (!conv[n]) all_conv = 0;
    }
    CK(cudaEventRecord(c->ev1, c->stream));
    CK(cudaEventSynchronize(c->ev1));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, c->ev0, c->ev1));
    for (int n = 0; n < nrhs; n++) infos[n].seconds = ms * 1e-3;
    for (int n = 0; n < nrhs; n++)
        if (broken[n])
            return fail(c, COLA_EINVAL, "cola_cg_solve_mrhs: BiCGStab broke down or met NaN/Inf in at least one system (<rhat, v>, <t, t> or rho vanished, or bad input); "
                                        "its x is the iterate of its last reliable update (see its info), the other systems were solved");
    if (!all_conv) return fail(c, COLA_ENOCONV, "cola_cg_solve_mrhs: max_iter reached before |r| <= tol*|b| for every system");
    return COLA_OK;
}

extern "C" {

cola_status cola_gauge_upload(cola_ctx *c, const double *host_links) { return gauge_upload_impl(c, host_links, 1); }
cola_status cola_gauge_upload_dev(cola_ctx *c, const double *dev_links) { return gauge_upload_impl(c, dev_links, 0); }

cola_status cola_gauge_info(const cola_ctx *c, double *max_unitarity_dev)
{
    if (!c || !max_unitarity_dev) return COLA_EINVAL;
    *max_unitarity_dev = c->max_unitarity_dev;
    return COLA_OK;
}

cola_status cola_gauge_info_r8(const cola_ctx *c, double *min_abs_u00)
{
    if (!c || !min_abs_u00) return COLA_EINVAL;
    *min_abs_u00 = sqrt(c->min_u00sq);
    return COLA_OK;
}

cola_status cola_clover_info(const cola_ctx *c, double *min_pivot)
{
    if (!c || !min_pivot) return COLA_EINVAL;
    *min_pivot = c->min_pivot;
    return COLA_OK;
}

cola_status cola_clover_unpack(cola_ctx *c, int which, void *canon_dev)
{
    ST(need_ready(c, "cola_clover_unpack"));
    if (!canon_dev) return fail(c, COLA_EINVAL, "cola_clover_unpack: NULL pointer");
    if (which == 0) CK(launch_clover_unpack(c->g, c->clovA64, 3, canon_dev, c->stream));
    else CK(launch_clover_unpack(c->g, c->clovI64, 2, canon_dev, c->stream));
    c->launches++;
    return COLA_OK;
}

cola_status cola_spinor_pack(cola_ctx *c, cola_prec prec, const void *canon_dev, void *internal_dev)
{
    if (!c) return COLA_EINVAL;
    if (!canon_dev || !internal_dev) return fail(c, COLA_EINVAL, "cola_spinor_pack: NULL pointer");
    if (prec != COLA_F64 && prec != COLA_F32) return fail(c, COLA_EINVAL, "cola_spinor_pack: prec must be COLA_F64 or COLA_F32 (COLA_F32_H16 uses fp32 spinors)");
    CK(launch_spinor_pack(prec, c->g, canon_dev, internal_dev, c->stream));
    c->launches++;
    return COLA_OK;
}

cola_status cola_spinor_unpack(cola_ctx *c, cola_prec prec, const void *internal_dev, void *canon_dev)
{
    if (!c) return COLA_EINVAL;
    if (!canon_dev || !internal_dev) return fail(c, COLA_EINVAL, "cola_spinor_unpack: NULL pointer");
    if (prec != COLA_F64 && prec != COLA_F32) return fail(c, COLA_EINVAL, "cola_spinor_unpack: prec must be COLA_F64 or COLA_F32 (COLA_F32_H16 uses fp32 spinors)");
    CK(launch_spinor_unpack(prec, c->g, internal_dev, canon_dev, c->stream));
    c->launches++;
    return COLA_OK;
}

cola_status cola_spinor_convert(cola_ctx *c, cola_prec dst_prec, const void *src_dev, void *dst_dev, int n_half)
{
    if (!c) return COLA_EINVAL;
    if (!src_dev || !dst_dev || n_half < 1 || n_half > 2) return fail(c, COLA_EINVAL, "cola_spinor_convert: bad argument");
    if (dst_prec != COLA_F64 && dst_prec != COLA_F32) return fail(c, COLA_EINVAL, "cola_spinor_convert: dst_prec must be COLA_F64 or COLA_F32");
    const cola_prec src_prec = dst_prec == COLA_F64 ? COLA_F32 : COLA_F64;
    for (int h = 0; h < n_half; h++) {
        CK(launch_spinor_convert(dst_prec, (const char *)src_dev + h * half_bytes(c, src_prec), (char *)dst_dev + h * half_bytes(c, dst_prec), c->Vh, c->stream));
        c->launches++;
    }
    return COLA_OK;
}

cola_status cola_dslash_apply(cola_ctx *c, cola_prec prec, cola_parity out_parity, const void *in_dev, void *out_dev)
{
    ST(need_ready(c, "cola_dslash_apply"));
    if (!in_dev || !out_dev || in_dev == out_dev) return fail(c, COLA_EINVAL, "cola_dslash_apply: NULL or aliased buffers");
    if (out_parity != COLA_EVEN && out_parity != COLA_ODD) return fail(c, COLA_EINVAL, "cola_dslash_apply: bad parity");
    return dslash(c, prec, (int)out_parity, 0, in_dev, out_dev, nullptr, 0, 0.0, 0, nullptr, 0);
}

cola_status cola_fermion_matrix_apply(cola_ctx *c, cola_prec prec, int dagger, const void *in_full_dev, void *out_full_dev)
{
    ST(need_ready(c, "cola_fermion_matrix_apply"));
    if (!in_full_dev || !out_full_dev || in_full_dev == out_full_dev) return fail(c, COLA_EINVAL, "cola_fermion_matrix_apply: NULL or aliased buffers");
    return fmatrix(c, prec, dagger ? 1 : 0, in_full_dev, out_full_dev, nullptr);
}

cola_status cola_schur_apply(cola_ctx *c, cola_prec prec, int dagger, const void *in_even_dev, void *out_even_dev)
{
    ST(need_ready(c, "cola_schur_apply"));
    if (!in_even_dev || !out_even_dev || in_even_dev == out_even_dev) return fail(c, COLA_EINVAL, "cola_schur_apply: NULL or aliased buffers");
    return schur(c, prec, dagger ? 1 : 0, in_even_dev, out_even_dev, nullptr);
}

cola_status cola_spinor_norm2(cola_ctx *c, cola_prec prec, const void *v_dev, int n_half, double *out_dev)
{
    if (!c) return COLA_EINVAL;
    if (!c->ws) return fail(c, COLA_ENOTREADY, "cola_spinor_norm2: no workspace (call cola_set_workspace)");
    if (prec != COLA_F64 && prec != COLA_F32) return fail(c, COLA_EINVAL, "cola_spinor_norm2: prec must be COLA_F64 or COLA_F32");
    if (!v_dev || !out_dev || (n_half != 1 && n_half != 2)) return fail(c, COLA_EINVAL, "cola_spinor_norm2: NULL pointer or n_half not 1 / 2");
    return norm2(c, prec, v_dev, (size_t)n_half * c->Vh, out_dev);
}

cola_status cola_cg_solve(cola_ctx *c, const cola_solve_params *sp, const void *b_canon_dev, void *x_canon_dev, cola_solve_info *info)
{
    return solve_impl(c, sp, b_canon_dev, x_canon_dev, info);
}

cola_status cola_cg_solve_history(cola_ctx *c, const cola_solve_params *sp, const void *b_canon_dev, void *x_canon_dev, cola_solve_info *info,
                                  double *resid_hist_host, int hist_len, int *update_iters_host, int update_len)
{
    if (!c) return COLA_EINVAL;
    if (!resid_hist_host || hist_len < 1) return fail(c, COLA_EINVAL, "cola_cg_solve_history: NULL or empty history buffer");
    if (update_iters_host && update_len < 1) return fail(c, COLA_EINVAL, "cola_cg_solve_history: empty update buffer");
    c->hist = resid_hist_host;
    c->hist_len = hist_len;
    c->upd_iters = update_iters_host;
    c->upd_len = update_iters_host ? update_len : 0;
    const cola_status st = solve_impl(c, sp, b_canon_dev, x_canon_dev, info);
    c->hist = nullptr;
    c->hist_len = 0;
    c->upd_iters = nullptr;
    c->upd_len = 0;
    return st;
}

// ---- end-to-end variants with HOST buffers.  Staging lives in the tail of the solver scratch
// (the solver uses at most 10 of its 12 half-vector slots when it is called from here; the two
// canonical staging buffers below need 2 full fp64 vectors = 4 slots, so operators stage in the
// first slots and the solve stages in x/b of the caller through the separate tmp region).
static cola_status host_op(cola_ctx *c, cola_prec prec, int which, int arg, const void *in_host, void *out_host)
{
    ST(need_ready(c, "cola_*_apply_host"));
    if (!in_host || !out_host) return fail(c, COLA_EINVAL, "cola_*_apply_host: NULL pointer");
    CK(cudaSetDevice(c->p.device));
    const size_t fb = 2 * half_bytes(c, prec);
    char *canon = c->scratch, *in_int = canon + fb, *out_int = in_int + fb;
    CK(cudaMemcpyAsync(canon, in_host, fb, cudaMemcpyHostToDevice, c->stream));
    CK(launch_spinor_pack(prec, c->g, canon, in_int, c->stream));
    c->launches++;
    if (which == 0) {
        const int p = arg;
        const size_t hb = half_bytes(c, prec);
        CK(cudaMemsetAsync(out_int, 0, fb, c->stream));
        ST(dslash(c, prec, p, 0, in_int + (1 - p) * hb, out_int + p * hb, nullptr, 0, 0.0, 0, nullptr, 0));
    } else {
        ST(fmatrix(c, prec, arg, in_int, out_int, nullptr));
    }
    CK(launch_spinor_unpack(prec, c->g, out_int, canon, c->stream));
    c->launches++;
    CK(cudaMemcpyAsync(out_host, canon, fb, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return COLA_OK;
}

cola_status cola_dslash_apply_host(cola_ctx *c, cola_prec prec, cola_parity out_parity, const void *in_canon_host, void *out_canon_host)
{
    if (c && out_parity != COLA_EVEN && out_parity != COLA_ODD) return fail(c, COLA_EINVAL, "cola_dslash_apply_host: bad parity");
    return host_op(c, prec, 0, (int)out_parity, in_canon_host, out_canon_host);
}

cola_status cola_fermion_matrix_apply_host(cola_ctx *c, cola_prec prec, int dagger, const void *in_canon_host, void *out_canon_host)
{
    return host_op(c, prec, 1, dagger ? 1 : 0, in_canon_host, out_canon_host);
}

cola_status cola_cg_solve_host(cola_ctx *c, const cola_solve_params *sp, const void *b_canon_host, void *x_canon_host, cola_solve_info *info)
{
    ST(need_ready(c, "cola_cg_solve_host"));
    if (!b_canon_host || !x_canon_host) return fail(c, COLA_EINVAL, "cola_cg_solve_host: NULL pointer");
    CK(cudaSetDevice(c->p.device));
    // canonical staging inside the solver's own scratch (solve_impl: packed source B = slots 0-1, solution X = slots 2-3):
    // the canonical b is staged in X's slots -- it is packed into B before X is zeroed -- and the canonical x is
    // unpacked over B, which is dead once the true residual has been formed.  No mode needs extra room.
    const size_t fb = 2 * half_bytes(c, COLA_F64);
    char *stage_b = c->scratch + fb, *stage_x = c->scratch;
    if (!sp) return fail(c, COLA_EINVAL, "cola_cg_solve_host: NULL solve parameters");
    CK(cudaMemcpyAsync(stage_b, b_canon_host, fb, cudaMemcpyHostToDevice, c->stream));
    cola_status st = solve_impl(c, sp, stage_b, stage_x, info);
    if (st != COLA_OK && st != COLA_ENOCONV) return st;
    CK(cudaMemcpyAsync(x_canon_host, stage_x, fb, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return st;
}

// ---- multi-right-hand-side entry points
size_t cola_mrhs_workspace_bytes(const cola_ctx *c, int nrhs, int for_solver)
{
    if (!c || nrhs < 1 || nrhs > MRHS_MAX) return 0;
    const CarveM k = carve_m(c, nrhs);
    return for_solver ? k.total : k.op_total;
}

cola_status cola_set_mrhs_workspace(cola_ctx *c, void *dev_ptr, size_t bytes, int nrhs)
{
    if (!c) return COLA_EINVAL;
    c->m_nrhs = 0;
    if (!dev_ptr && nrhs == 0) return COLA_OK;   // release
    if (nrhs < 1 || nrhs > MRHS_MAX) return fail(c, COLA_EINVAL, "cola_set_mrhs_workspace: nrhs must be 1..16");
    if (!dev_ptr || ((uintptr_t)dev_ptr & 255)) return fail(c, COLA_EINVAL, "cola_set_mrhs_workspace: pointer must be non-NULL and 256-byte aligned");
    const CarveM k = carve_m(c, nrhs);
    if (bytes < k.op_total) return fail(c, COLA_ENOMEM, "cola_set_mrhs_workspace: workspace smaller than cola_mrhs_workspace_bytes()");
    c->m_solver = bytes >= k.total;   // room for the batched solver's vectors as well
    char *w = (char *)dev_ptr;
    c->m_tmp32 = w + k.tmp32; c->m_r64 = w + k.r64; c->m_rhs = w + k.rhs; c->m_qs = w + k.qs;
    c->m_x32 = w + k.x32; c->m_r32 = w + k.r32; c->m_p32 = w + k.p32; c->m_q32 = w + k.q32;
    c->m_rhat32 = w + k.rhat32;
    c->m_ctlb = (CtlB *)(w + k.ctlb);
    c->m_statb = (HostStatus *)(w + k.ctlb + MRHS_MAX * sizeof(CtlB));
    c->m_tt = (double *)(w + k.ctlb + MRHS_MAX * (sizeof(CtlB) + sizeof(HostStatus)));
    c->m_partials = (double *)(w + k.partials);
    c->m_nsb = k.nsb;
    c->m_nrhs = nrhs;
    return COLA_OK;
}

static MrhsList identity_list(int nrhs)
{
    int v[MRHS_MAX];
    for (int k = 0; k < MRHS_MAX; k++) v[k] = k;
    return list_of(v, nrhs);
}

cola_status cola_dslash_apply_mrhs(cola_ctx *c, cola_prec prec, cola_parity out_parity, int nrhs, const void *in_dev, void *out_dev)
{
    ST(need_mrhs(c, "cola_dslash_apply_mrhs", nrhs));
    if (!in_dev || !out_dev || in_dev == out_dev) return fail(c, COLA_EINVAL, "cola_dslash_apply_mrhs: NULL or aliased buffers");
    if (out_parity != COLA_EVEN && out_parity != COLA_ODD) return fail(c, COLA_EINVAL, "cola_dslash_apply_mrhs: bad parity");
    const size_t hb = half_bytes(c, prec);
    return dslash_m(c, prec, (int)out_parity, 0, identity_list(nrhs), nrhs, in_dev, hb, out_dev, hb, nullptr, 0, 0, 0.0, 0, nullptr, 0, nullptr);
}

cola_status cola_fermion_matrix_apply_mrhs(cola_ctx *c, cola_prec prec, int dagger, int nrhs, const void *in_full_dev, void *out_full_dev)
{
    ST(need_mrhs(c, "cola_fermion_matrix_apply_mrhs", nrhs));
    if (!in_full_dev || !out_full_dev || in_full_dev == out_full_dev) return fail(c, COLA_EINVAL, "cola_fermion_matrix_apply_mrhs: NULL or aliased buffers");
    const size_t hb = half_bytes(c, prec), fb = 2 * hb;
    const char *in_e = (const char *)in_full_dev, *in_o = in_e + hb;
    char *out_e = (char *)out_full_dev, *out_o = out_e + hb;
    const MrhsList L = identity_list(nrhs);
    const int dg = dagger ? 1 : 0;
    ST(dslash_m(c, prec, 0, dg, L, nrhs, in_o, fb, out_e, fb, in_e, fb, 1, -c->p.kappa, 0, nullptr, 0, nullptr));
    ST(dslash_m(c, prec, 1, dg, L, nrhs, in_e, fb, out_o, fb, in_o, fb, 1, -c->p.kappa, 0, nullptr, 0, nullptr));
    return COLA_OK;
}

cola_status cola_schur_apply_mrhs(cola_ctx *c, cola_prec prec, int dagger, int nrhs, const void *in_even_dev, void *out_even_dev)
{
    ST(need_mrhs(c, "cola_schur_apply_mrhs", nrhs));
    if (!in_even_dev || !out_even_dev || in_even_dev == out_even_dev) return fail(c, COLA_EINVAL, "cola_schur_apply_mrhs: NULL or aliased buffers");
    const size_t hb = half_bytes(c, prec);
    return schur_m(c, prec, dagger ? 1 : 0, identity_list(nrhs), nrhs, in_even_dev, hb, prec == COLA_F64 ? c->m_r64 : c->m_tmp32, out_even_dev, hb, nullptr, nullptr);
}

cola_status cola_cg_solve_mrhs(cola_ctx *c, const cola_solve_params *sp, int nrhs, const void *b_canon_dev, void *x_canon_dev, cola_solve_info *infos)
{
    return solve_mrhs_impl(c, sp, nrhs, b_canon_dev, x_canon_dev, infos);
}

// Host-side self-test of the index machinery the kernels rely on (no GPU needed): magic-number division against the
// hardware division, tile shapes and sweep descriptors against their invariants.
cola_status cola_selftest_host(char *msg, size_t msg_len)
{
    auto say = [&](const char *what, long a, long b) {
        if (msg && msg_len) snprintf(msg, msg_len, "%s (%ld, %ld)", what, a, b);
        return COLA_EINVAL;
    };
    // floor(n/d) for every divisor up to 4096 (and a few large ones) over a spread of n < 2^31 incl. the edges
    unsigned long long lcg = 88172645463325252ull;
    for (unsigned d = 1; d <= 4200; d++) {
        const FastDiv f = make_fastdiv(d);
        auto q = [&](unsigned n) { return f.d == 1u ? n : (unsigned)(((unsigned long long)n * f.m) >> 32) >> f.sh; };
        const unsigned edge[] = {0u, 1u, d - 1u, d, d + 1u, 2u * d - 1u, 2u * d, 0x7fffffffu, 0x7ffffffeu, 0x7fffffffu / d * d, 0x7fffffffu / d * d - 1u};
        for (unsigned n : edge)
            if (n <= 0x7fffffffu && q(n) != n / d) return say("fastdiv edge", (long)n, (long)d);
        for (int k = 0; k < 2000; k++) {
            lcg = lcg * 6364136223846793005ull + 1442695040888963407ull;
            const unsigned n = (unsigned)(lcg >> 33);
            if (q(n) != n / d) return say("fastdiv", (long)n, (long)d);
        }
    }
    for (unsigned d : {65536u, 1000003u, 16777216u, 0x40000000u, 0x7fffffffu}) {
        const FastDiv f = make_fastdiv(d);
        for (unsigned n : {0u, d - 1u, d, d + 1u, 0x7fffffffu})
            if ((f.d == 1u ? n : (unsigned)(((unsigned long long)n * f.m) >> 32) >> f.sh) != n / d) return say("fastdiv large", (long)n, (long)d);
    }
    // tiles and sweeps on a spread of lattices
    const int L[][4] = {{2, 2, 2, 2}, {4, 4, 4, 4}, {4, 2, 6, 2}, {12, 10, 6, 4}, {16, 16, 16, 32}, {32, 32, 32, 64}, {48, 48, 48, 96}, {64, 64, 64, 128}, {6, 4, 2, 8}, {128, 2, 2, 2}};
    for (const auto &d : L) {
        Geom g;
        memset(&g, 0, sizeof(g));
        g.X = d[0]; g.Y = d[1]; g.Z = d[2]; g.T = d[3]; g.Xh = d[0] / 2;
        g.Vh = g.Xh * g.Y * g.Z * g.T;
        for (int ms : {32, 64, 128, 256}) {
            const Tile t = make_tile(g, ms, 16);
            const int ext[4] = {g.Xh, g.Y, g.Z, g.T};
            int vol = 1;
            for (int k = 0; k < 4; k++) {
                if (ext[k] % (1 << t.sh[k])) return say("tile extent does not divide the lattice", d[k], 1 << t.sh[k]);
                vol <<= t.sh[k];
            }
            if (vol != t.vol || vol > ms || t.ntiles * vol != g.Vh) return say("tile volume", vol, ms);
        }
        for (size_t budget : {(size_t)1, (size_t)100000, (size_t)40 << 20}) {
            for (int mult : {1, 2}) {
                const int zb = choose_zband(g.Xh * g.Y, g.Z, 96, budget, mult);
                if (zb < 0 || zb >= g.Z + (zb == 0) || (zb && (g.Z % zb || zb % mult))) return say("zband", zb, g.Z);
                const Sweep w = make_sweep(g, zb);
                if (w.on && ((g.Xh * g.Y) % 64 || g.Z % w.zb)) return say("sweep on unsuitable geometry", zb, g.Z);
                if (w.on) {   // the block permutation is a bijection on [0, Vh/64)
                    const unsigned nb = (unsigned)(g.Vh / 64), up = w.d_up.d;
                    unsigned long long sum = 0, want = (unsigned long long)nb * (nb - 1) / 2;
                    for (unsigned b = 0; b < nb; b++) {
                        const unsigned q1 = b / up, u = b % up, q2 = q1 / (unsigned)w.zb, zi = q1 % (unsigned)w.zb, band = q2 / (unsigned)g.T, t = q2 % (unsigned)g.T;
                        const unsigned run = ((t * (unsigned)g.Z + band * (unsigned)w.zb + zi) * up) + u;
                        if (run >= nb) return say("sweep run out of range", (long)run, (long)nb);
                        sum += run;
                    }
                    if (sum != want) return say("sweep is not a permutation", (long)sum, (long)want);
                }
            }
        }
    }
    if (msg && msg_len) snprintf(msg, msg_len, "ok");
    return COLA_OK;
}

unsigned long long cola_launch_count(const cola_ctx *c) { return c ? c->launches : 0; }

}  // extern "C"
