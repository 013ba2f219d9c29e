// cola_blas.cu -- fused BLAS-1 layer of the CGLS iteration.
// Vectors are flat arrays of 16-byte chunks; alpha and beta are formed on the device from the
// reduction results in Ctl, so no scalar crosses the PCIe bus inside an iteration.  Reductions are
// accumulated in fp64 also for fp32 vectors and are deterministic (fixed grid, fixed order).
#include "cola_device.cuh"

namespace cola {

namespace {

constexpr int BB = 256;
constexpr int MAX_BLOCKS = 148 * 8;

inline unsigned blas_grid(size_t n_chunks)
{
    size_t b = (n_chunks + BB - 1) / BB;
    return (unsigned)(b < (size_t)MAX_BLOCKS ? b : (size_t)MAX_BLOCKS);
}

__device__ __forceinline__ double sq(const float4 &v) { return (double)(v.x * v.x + v.y * v.y) + (double)(v.z * v.z + v.w * v.w); }
__device__ __forceinline__ double sq(const double2 &v) { return v.x * v.x + v.y * v.y; }
__device__ __forceinline__ float4 axpy(float a, const float4 &x, const float4 &y) { return make_float4(y.x + a * x.x, y.y + a * x.y, y.z + a * x.z, y.w + a * x.w); }
__device__ __forceinline__ double2 axpy(double a, const double2 &x, const double2 &y) { return make_double2(y.x + a * x.x, y.y + a * x.y); }

template <typename T>
__global__ void __launch_bounds__(BB) norm2_kernel(const typename VT<T>::V *v, size_t n, ReduceWs red, unsigned *counter, double *out)
{
    double acc = 0.0;
    for (size_t k = (size_t)blockIdx.x * BB + threadIdx.x; k < n; k += (size_t)gridDim.x * BB) acc += sq(v[k]);
    grid_sum_finalize(acc, red, counter, out);
}

// r -= alpha q, alpha = gamma / qq;  rr = |r|^2
template <typename T>
__global__ void __launch_bounds__(BB) r_update_kernel(typename VT<T>::V *r, const typename VT<T>::V *q, Ctl *ctl, int cur, int iter, const int *skip, HostStatus *mirror, size_t n, ReduceWs red)
{
    pdl_trigger();
    pdl_wait();
    if (skip && *skip) return;
    const T ma = (T)(-(ctl->gam[cur] / ctl->qq));
    double acc = 0.0;
    for (size_t k = (size_t)blockIdx.x * BB + threadIdx.x; k < n; k += (size_t)gridDim.x * BB) {
        const typename VT<T>::V v = axpy(ma, q[k], r[k]);
        r[k] = v;
        acc += sq(v);
    }
    double rr;
    if (grid_sum_last(acc, red, &ctl->counter[1], &rr)) {
        ctl->rr = rr;
        ctl->iters = iter;
        const double rmax2 = fmax(ctl->rmax2, rr);
        ctl->rmax2 = rmax2;
        const int flag = (rr <= ctl->target2 || rr < ctl->delta2 * rmax2) ? 1 : 0;
        if (flag) ctl->flag = 1;
        if (mirror) {   // publish to the host without a DMA copy in the stream
            volatile HostStatus *m = mirror;
            m->rr = rr;
            m->flag = flag;
            __threadfence_system();
            m->iters = iter;
        }
    }
}

// x += alpha p (DO_X);  p = s + beta p (DO_P);  alpha = gamma/qq, beta = gamma_new/gamma
template <typename T, bool DO_X, bool DO_P>
__global__ void __launch_bounds__(BB) xp_update_kernel(typename VT<T>::V *x, typename VT<T>::V *p, const typename VT<T>::V *s, const Ctl *ctl, int cur, const int *skip, size_t n)
{
    pdl_trigger();
    pdl_wait();
    if (skip && *skip) return;
    const T alpha = (T)(ctl->gam[cur] / ctl->qq);
    const T beta = (T)(ctl->gam[cur ^ 1] / ctl->gam[cur]);
    for (size_t k = (size_t)blockIdx.x * BB + threadIdx.x; k < n; k += (size_t)gridDim.x * BB) {
        const typename VT<T>::V pv = p[k];
        if (DO_X) x[k] = axpy(alpha, pv, x[k]);
        if (DO_P) p[k] = axpy(beta, pv, s[k]);
    }
}

// out64 = a*A + b*B; optional fp32 copy (internal fp32 layout needs chunk pairing, so this kernel works
// per site-chunk pair: thread handles double2 chunks 2k, 2k+1 of site i = one float4 chunk k)
__global__ void __launch_bounds__(BB) axpby64_kernel(double2 *out, double a, const double2 *A, double b, const double2 *B, float4 *out32,
                                                     size_t n_sites, ReduceWs red, unsigned *counter, double *norm_out)
{
    double acc = 0.0;
    const size_t n = 6 * n_sites;
    for (size_t tid = (size_t)blockIdx.x * BB + threadIdx.x; tid < n; tid += (size_t)gridDim.x * BB) {
        const size_t k = tid / n_sites, i = tid - k * n_sites;
        const size_t c0 = (2 * k) * n_sites + i, c1 = (2 * k + 1) * n_sites + i;
        double2 v0, v1;
        if (B) {
            const double2 a0 = A[c0], a1 = A[c1], b0 = B[c0], b1 = B[c1];
            v0 = make_double2(a * a0.x + b * b0.x, a * a0.y + b * b0.y);
            v1 = make_double2(a * a1.x + b * b1.x, a * a1.y + b * b1.y);
        } else {
            const double2 a0 = A[c0], a1 = A[c1];
            v0 = make_double2(a * a0.x, a * a0.y);
            v1 = make_double2(a * a1.x, a * a1.y);
        }
        if (out) {
            out[c0] = v0;
            out[c1] = v1;
        }
        if (out32) out32[k * n_sites + i] = make_float4((float)v0.x, (float)v0.y, (float)v1.x, (float)v1.y);
        acc += sq(v0) + sq(v1);
    }
    if (red.partials) grid_sum_finalize(acc, red, counter, norm_out);
}

// x64 += x32; x32 = 0
__global__ void __launch_bounds__(BB) accumulate_kernel(double2 *x64, float4 *x32, size_t n_sites)
{
    const size_t n = 6 * n_sites;
    for (size_t tid = (size_t)blockIdx.x * BB + threadIdx.x; tid < n; tid += (size_t)gridDim.x * BB) {
        const size_t k = tid / n_sites, i = tid - k * n_sites;
        const size_t c0 = (2 * k) * n_sites + i, c1 = (2 * k + 1) * n_sites + i;
        const float4 v = x32[k * n_sites + i];
        double2 a0 = x64[c0], a1 = x64[c1];
        a0.x += v.x; a0.y += v.y; a1.x += v.z; a1.y += v.w;
        x64[c0] = a0;
        x64[c1] = a1;
        x32[k * n_sites + i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

// ---- BiCGStab.  A float4 chunk holds two complex numbers, a double2 chunk one; alpha, omega, beta
// are formed in fp64 from the device-resident dots (CtlB) by every thread and applied in the vectors' precision.
struct Cx { double re, im; };
__device__ __forceinline__ Cx cdiv(const double (&a)[2], const double (&b)[2])
{
    const double d = b[0] * b[0] + b[1] * b[1];
    return Cx{(a[0] * b[0] + a[1] * b[1]) / d, (a[1] * b[0] - a[0] * b[1]) / d};
}
__device__ __forceinline__ Cx cmul(Cx a, Cx b) { return Cx{a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
// y + c x on a chunk (complex scalar c)
__device__ __forceinline__ float4 caxpy(float cr, float ci, const float4 &x, const float4 &y)
{
    return make_float4(y.x + cr * x.x - ci * x.y, y.y + cr * x.y + ci * x.x, y.z + cr * x.z - ci * x.w, y.w + cr * x.w + ci * x.z);
}
__device__ __forceinline__ double2 caxpy(double cr, double ci, const double2 &x, const double2 &y)
{
    return make_double2(y.x + cr * x.x - ci * x.y, y.y + cr * x.y + ci * x.x);
}
// sum conj(a) b over a chunk, added to (re, im)
__device__ __forceinline__ void cdot_acc(const float4 &a, const float4 &b, double &re, double &im)
{
    re += (double)(a.x * b.x + a.y * b.y + a.z * b.z + a.w * b.w);
    im += (double)(a.x * b.y - a.y * b.x + a.z * b.w - a.w * b.z);
}
__device__ __forceinline__ void cdot_acc(const double2 &a, const double2 &b, double &re, double &im)
{
    re += a.x * b.x + a.y * b.y;
    im += a.x * b.y - a.y * b.x;
}
// omega = <t, s> / <t, t>.  t = S s vanishes only with s (S is non-singular): the half step x + alpha p already solves the
// system exactly.  omega = 0 then completes the pass with x += alpha p, r = s = 0 instead of 0/0.
__device__ __forceinline__ Cx bicg_omega(const CtlB *ctl)
{
    if (ctl->tt == 0.0) return Cx{0.0, 0.0};
    return Cx{ctl->ts[0] / ctl->tt, ctl->ts[1] / ctl->tt};
}
// beta = (rho_next / rho) (alpha / omega), alpha = rho / rv  =>  beta = rho_next / (rv omega)
__device__ __forceinline__ void bicg_set_beta(CtlB *ctl, const double (&rho_next)[2])
{
    const Cx om = bicg_omega(ctl);
    const Cx den = cmul(Cx{ctl->rv[0], ctl->rv[1]}, om);
    const double d[2] = {den.re, den.im};
    const Cx b = cdiv(rho_next, d);
    ctl->rho_next[0] = rho_next[0];
    ctl->rho_next[1] = rho_next[1];
    ctl->beta[0] = b.re;
    ctl->beta[1] = b.im;
}

template <typename T>
__global__ void __launch_bounds__(BB) bicg_dot_kernel(const typename VT<T>::V *a, const typename VT<T>::V *b, CtlB *ctl, int which, const int *skip, size_t n, ReduceWs red)
{
    pdl_trigger();
    pdl_wait();
    if (skip && *skip) return;
    double v[2] = {0.0, 0.0};
    for (size_t k = (size_t)blockIdx.x * BB + threadIdx.x; k < n; k += (size_t)gridDim.x * BB) cdot_acc(a[k], b[k], v[0], v[1]);
    double tot[2];
    if (grid_sum_last_n<2>(v, red, &ctl->counter[0], tot)) {
        if (which == 0) {
            ctl->rv[0] = tot[0]; ctl->rv[1] = tot[1];
            ctl->rho[0] = ctl->rho_next[0]; ctl->rho[1] = ctl->rho_next[1];
        } else if (which == 1) {
            ctl->ts[0] = tot[0]; ctl->ts[1] = tot[1];
        } else {
            bicg_set_beta(ctl, tot);
        }
    }
}

template <typename T>
__global__ void __launch_bounds__(BB) bicg_s_update_kernel(typename VT<T>::V *sv, const typename VT<T>::V *r, const typename VT<T>::V *v, const CtlB *ctl, const int *skip, size_t n)
{
    pdl_trigger();
    pdl_wait();
    if (skip && *skip) return;
    const Cx al = cdiv(ctl->rho, ctl->rv);
    const T mr = (T)(-al.re), mi = (T)(-al.im);
    for (size_t k = (size_t)blockIdx.x * BB + threadIdx.x; k < n; k += (size_t)gridDim.x * BB) sv[k] = caxpy(mr, mi, v[k], r[k]);
}

template <typename T>
__global__ void __launch_bounds__(BB) bicg_xr_update_kernel(typename VT<T>::V *x, typename VT<T>::V *r, const typename VT<T>::V *p, const typename VT<T>::V *sv,
                                                            const typename VT<T>::V *t, const typename VT<T>::V *rhat, CtlB *ctl, int iter, const int *skip,
                                                            HostStatus *mirror, size_t n, ReduceWs red)
{
    pdl_trigger();
    pdl_wait();
    if (skip && *skip) return;
    const Cx al = cdiv(ctl->rho, ctl->rv), om = bicg_omega(ctl);
    const T ar = (T)al.re, ai = (T)al.im, wr = (T)om.re, wi = (T)om.im;
    double v[3] = {0.0, 0.0, 0.0};
    for (size_t k = (size_t)blockIdx.x * BB + threadIdx.x; k < n; k += (size_t)gridDim.x * BB) {
        const typename VT<T>::V s_ = sv[k];
        x[k] = caxpy(wr, wi, s_, caxpy(ar, ai, p[k], x[k]));
        const typename VT<T>::V rn = caxpy(-wr, -wi, t[k], s_);
        r[k] = rn;
        v[0] += sq(rn);
        cdot_acc(rhat[k], rn, v[1], v[2]);
    }
    double tot[3];
    if (grid_sum_last_n<3>(v, red, &ctl->counter[1], tot)) {
        const double rr = tot[0];
        const double rho_next[2] = {tot[1], tot[2]};
        bicg_set_beta(ctl, rho_next);
        ctl->rr = rr;
        ctl->iters = iter;
        const double rmax2 = fmax(ctl->rmax2, rr);
        ctl->rmax2 = rmax2;
        const int flag = (rr <= ctl->target2 || rr < ctl->delta2 * rmax2) ? 1 : 0;
        if (flag) ctl->flag = 1;
        if (mirror) {
            volatile HostStatus *m = mirror;
            m->rr = rr;
            m->flag = flag;
            __threadfence_system();
            m->iters = iter;
        }
    }
}

template <typename T>
__global__ void __launch_bounds__(BB) bicg_p_update_kernel(typename VT<T>::V *p, const typename VT<T>::V *r, const typename VT<T>::V *v, const CtlB *ctl, const int *skip, size_t n)
{
    pdl_trigger();
    pdl_wait();
    if (skip && *skip) return;
    const Cx om = bicg_omega(ctl);
    const T br = (T)ctl->beta[0], bi = (T)ctl->beta[1], mwr = (T)(-om.re), mwi = (T)(-om.im);
    for (size_t k = (size_t)blockIdx.x * BB + threadIdx.x; k < n; k += (size_t)gridDim.x * BB) p[k] = caxpy(br, bi, caxpy(mwr, mwi, v[k], p[k]), r[k]);
}

// ---- batched (multi-right-hand-side) variants: blockIdx.y = position in the list, same arithmetic per vector
inline unsigned mrhs_grid(size_t n_chunks)
{
    size_t b = (n_chunks + BB - 1) / BB;
    return (unsigned)(b < (size_t)(MAX_BLOCKS / 4) ? b : (size_t)(MAX_BLOCKS / 4));
}

template <typename T>
__global__ void __launch_bounds__(BB) r_update_mrhs_kernel(char *r0, const char *q0, size_t stride, const CtlM *ctl, int cur, const __grid_constant__ MrhsList list,
                                                           const int *skip, size_t n, double *partials)
{
    typedef typename VT<T>::V V;
    if (skip && *skip) return;
    __shared__ double sm[33];
    const int vec = list.v[blockIdx.y];
    V *r = reinterpret_cast<V *>(r0 + (size_t)vec * stride);
    const V *q = reinterpret_cast<const V *>(q0 + (size_t)vec * stride);
    const T ma = (T)(-(ctl->gam[cur][vec] / ctl->qq[vec]));
    double acc = 0.0;
    for (size_t k = (size_t)blockIdx.x * BB + threadIdx.x; k < n; k += (size_t)gridDim.x * BB) {
        const V v = axpy(ma, q[k], r[k]);
        r[k] = v;
        acc += sq(v);
    }
    acc = block_sum(acc, sm);
    if (threadIdx.x == 0) partials[(size_t)vec * gridDim.x + blockIdx.x] = acc;
}

// one block, one thread per list entry: rmax2, trigger, flag, host mirror
__global__ void __launch_bounds__(32) decide_mrhs_kernel(CtlM *ctl, const __grid_constant__ MrhsList list, int nrhs, int iter, const int *skip, HostStatusM *mirror)
{
    if (skip && *skip) return;
    const int k = threadIdx.x;
    bool trig = false;
    int vec = 0;
    double rr = 0.0;
    if (k < nrhs) {
        vec = list.v[k];
        rr = ctl->rr[vec];
        const double rmax2 = fmax(ctl->rmax2[vec], rr);
        ctl->rmax2[vec] = rmax2;
        trig = rr <= ctl->target2[vec] || rr < ctl->delta2 * rmax2;
    }
    unsigned mask = 0;
    for (int j = 0; j < 32; j++) {
        const int tj = __shfl_sync(0xffffffffu, trig ? 1 : 0, j);
        const int vj = __shfl_sync(0xffffffffu, vec, j);
        if (tj) mask |= 1u << vj;
    }
    if (mirror && k < nrhs) (reinterpret_cast<volatile double *>(mirror->rr))[vec] = rr;
    __syncwarp();
    if (k == 0) {
        ctl->iters = iter;
        ctl->trig = mask;
        if (mask) ctl->flag = 1;
        if (mirror) {
            volatile HostStatusM *m = mirror;
            m->trig = mask;
            m->flag = mask ? 1 : 0;
            __threadfence_system();
            m->iters = iter;
        }
    }
}

template <typename T, bool DO_X, bool DO_P>
__global__ void __launch_bounds__(BB) xp_update_mrhs_kernel(char *x0, char *p0, const char *s0, size_t stride, const CtlM *ctl, int cur, const __grid_constant__ MrhsList list,
                                                            const int *skip, size_t n)
{
    typedef typename VT<T>::V V;
    if (skip && *skip) return;
    const int vec = list.v[blockIdx.y];
    V *x = reinterpret_cast<V *>(x0 + (size_t)vec * stride);
    V *p = reinterpret_cast<V *>(p0 + (size_t)vec * stride);
    const V *s = reinterpret_cast<const V *>(s0 + (size_t)vec * stride);
    const T alpha = (T)(ctl->gam[cur][vec] / ctl->qq[vec]);
    const T beta = (T)(ctl->gam[cur ^ 1][vec] / ctl->gam[cur][vec]);
    for (size_t k = (size_t)blockIdx.x * BB + threadIdx.x; k < n; k += (size_t)gridDim.x * BB) {
        const V pv = p[k];
        if (DO_X) x[k] = axpy(alpha, pv, x[k]);
        if (DO_P) p[k] = axpy(beta, pv, s[k]);
    }
}

}  // namespace

int blas_max_blocks() { return MAX_BLOCKS; }

int blas_mrhs_blocks(size_t n_sites, cola_prec prec) { return (int)mrhs_grid((prec == COLA_F64 ? 12 : 6) * n_sites); }

cudaError_t launch_r_update_mrhs(cola_prec prec, void *r, const void *q, size_t stride, const CtlM *ctl, int cur, const MrhsList &list, int nrhs,
                                 const int *skip, size_t n_sites, double *partials, cudaStream_t s)
{
    const size_t n = (prec == COLA_F64 ? 12 : 6) * n_sites;
    const dim3 grid(mrhs_grid(n), nrhs);
    if (prec == COLA_F64) r_update_mrhs_kernel<double><<<grid, BB, 0, s>>>((char *)r, (const char *)q, stride, ctl, cur, list, skip, n, partials);
    else r_update_mrhs_kernel<float><<<grid, BB, 0, s>>>((char *)r, (const char *)q, stride, ctl, cur, list, skip, n, partials);
    return cudaGetLastError();
}

cudaError_t launch_decide_mrhs(CtlM *ctl, const MrhsList &list, int nrhs, int iter, const int *skip, HostStatusM *mirror, cudaStream_t s)
{
    decide_mrhs_kernel<<<1, 32, 0, s>>>(ctl, list, nrhs, iter, skip, mirror);
    return cudaGetLastError();
}

cudaError_t launch_xp_update_mrhs(cola_prec prec, void *x, void *p, const void *sv, size_t stride, const CtlM *ctl, int cur, const MrhsList &list, int nrhs,
                                  int do_x, int do_p, const int *skip, size_t n_sites, cudaStream_t s)
{
    const size_t n = (prec == COLA_F64 ? 12 : 6) * n_sites;
    const dim3 grid(mrhs_grid(n), nrhs);
    char *x0 = (char *)x, *p0 = (char *)p;
    const char *s0 = (const char *)sv;
#define COLA_XP(T, X, P) xp_update_mrhs_kernel<T, X, P><<<grid, BB, 0, s>>>(x0, p0, s0, stride, ctl, cur, list, skip, n)
    if (prec == COLA_F64) {
        if (do_x && do_p) COLA_XP(double, true, true);
        else if (do_x) COLA_XP(double, true, false);
        else if (do_p) COLA_XP(double, false, true);
    } else {
        if (do_x && do_p) COLA_XP(float, true, true);
        else if (do_x) COLA_XP(float, true, false);
        else if (do_p) COLA_XP(float, false, true);
    }
#undef COLA_XP
    return cudaGetLastError();
}

#define COLA_BICG_DISPATCH(KERN, ...)                                                                                        \
    do {                                                                                                                   \
        if (prec == COLA_F64) {                                                                                            \
            typedef double2 V;                                                                                             \
            const size_t n = 12 * n_sites;                                                                                 \
            return launch_pdl(KERN<double>, dim3(blas_grid(n)), dim3(BB), s, __VA_ARGS__);                                 \
        } else {                                                                                                           \
            typedef float4 V;                                                                                              \
            const size_t n = 6 * n_sites;                                                                                  \
            return launch_pdl(KERN<float>, dim3(blas_grid(n)), dim3(BB), s, __VA_ARGS__);                                  \
        }                                                                                                                  \
    } while (0)

cudaError_t launch_bicg_dot(cola_prec prec, const void *a, const void *b, CtlB *ctl, int which, const int *skip, size_t n_sites, const ReduceWs &red, cudaStream_t s)
{
    COLA_BICG_DISPATCH(bicg_dot_kernel, (const V *)a, (const V *)b, ctl, which, skip, n, red);
}

cudaError_t launch_bicg_s_update(cola_prec prec, void *sv, const void *r, const void *v, const CtlB *ctl, const int *skip, size_t n_sites, cudaStream_t s)
{
    COLA_BICG_DISPATCH(bicg_s_update_kernel, (V *)sv, (const V *)r, (const V *)v, ctl, skip, n);
}

cudaError_t launch_bicg_xr_update(cola_prec prec, void *x, void *r, const void *p, const void *sv, const void *t, const void *rhat, CtlB *ctl, int iter,
                                  const int *skip, HostStatus *mirror, size_t n_sites, const ReduceWs &red, cudaStream_t s)
{
    COLA_BICG_DISPATCH(bicg_xr_update_kernel, (V *)x, (V *)r, (const V *)p, (const V *)sv, (const V *)t, (const V *)rhat, ctl, iter, skip, mirror, n, red);
}

cudaError_t launch_bicg_p_update(cola_prec prec, void *p, const void *r, const void *v, const CtlB *ctl, const int *skip, size_t n_sites, cudaStream_t s)
{
    COLA_BICG_DISPATCH(bicg_p_update_kernel, (V *)p, (const V *)r, (const V *)v, ctl, skip, n);
}
#undef COLA_BICG_DISPATCH

cudaError_t launch_norm2(cola_prec prec, const void *v, size_t n_sites, const ReduceWs &red, unsigned *counter, double *out, cudaStream_t s)
{
    if (prec == COLA_F64) {
        const size_t n = 12 * n_sites;
        norm2_kernel<double><<<blas_grid(n), BB, 0, s>>>((const double2 *)v, n, red, counter, out);
    } else {
        const size_t n = 6 * n_sites;
        norm2_kernel<float><<<blas_grid(n), BB, 0, s>>>((const float4 *)v, n, red, counter, out);
    }
    return cudaGetLastError();
}

cudaError_t launch_r_update(cola_prec prec, void *r, const void *q, Ctl *ctl, int cur, int iter, const int *skip, HostStatus *mirror, size_t n_sites, const ReduceWs &red, cudaStream_t s)
{
    if (prec == COLA_F64) {
        const size_t n = 12 * n_sites;
        return launch_pdl(r_update_kernel<double>, dim3(blas_grid(n)), dim3(BB), s, (double2 *)r, (const double2 *)q, ctl, cur, iter, skip, mirror, n, red);
    } else {
        const size_t n = 6 * n_sites;
        return launch_pdl(r_update_kernel<float>, dim3(blas_grid(n)), dim3(BB), s, (float4 *)r, (const float4 *)q, ctl, cur, iter, skip, mirror, n, red);
    }
    return cudaGetLastError();
}

template <typename T>
static void xp_dispatch(void *x, void *p, const void *sv, const Ctl *ctl, int cur, int do_x, int do_p, const int *skip, size_t n, cudaStream_t s)
{
    typedef typename VT<T>::V V;
    const unsigned grid = blas_grid(n);
    if (do_x && do_p) launch_pdl(xp_update_kernel<T, true, true>, dim3(grid), dim3(BB), s, (V *)x, (V *)p, (const V *)sv, ctl, cur, skip, n);
    else if (do_x) launch_pdl(xp_update_kernel<T, true, false>, dim3(grid), dim3(BB), s, (V *)x, (V *)p, (const V *)sv, ctl, cur, skip, n);
    else if (do_p) launch_pdl(xp_update_kernel<T, false, true>, dim3(grid), dim3(BB), s, (V *)x, (V *)p, (const V *)sv, ctl, cur, skip, n);
}

cudaError_t launch_xp_update(cola_prec prec, void *x, void *p, const void *sv, const Ctl *ctl, int cur, int do_x, int do_p, const int *skip, size_t n_sites, cudaStream_t s)
{
    if (prec == COLA_F64) xp_dispatch<double>(x, p, sv, ctl, cur, do_x, do_p, skip, 12 * n_sites, s);
    else xp_dispatch<float>(x, p, sv, ctl, cur, do_x, do_p, skip, 6 * n_sites, s);
    return cudaGetLastError();
}

cudaError_t launch_axpby64(void *out64, double a, const void *A64, double b, const void *B64, void *out32, size_t n_sites,
                           const ReduceWs *red, unsigned *counter, double *norm_out, cudaStream_t s)
{
    ReduceWs none = {nullptr, nullptr, nullptr};
    axpby64_kernel<<<blas_grid(6 * n_sites), BB, 0, s>>>((double2 *)out64, a, (const double2 *)A64, b, (const double2 *)B64, (float4 *)out32,
                                                        n_sites, red ? *red : none, counter, norm_out);
    return cudaGetLastError();
}

cudaError_t launch_accumulate(void *x64, void *x32, size_t n_sites, cudaStream_t s)
{
    accumulate_kernel<<<blas_grid(6 * n_sites), BB, 0, s>>>((double2 *)x64, (float4 *)x32, n_sites);
    return cudaGetLastError();
}

}  // namespace cola
