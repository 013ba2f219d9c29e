// cola_eig.cu -- vector kernels and the small dense eigen-solver of the low-mode solver (P:21
// "solvers for linear systems and eigenmodes", ref [1] P:65): thick-restart Lanczos on a Chebyshev polynomial of
// H = S^+ S (the driver is cola_eig_lowest in cola_api.cu).  All vectors are fp64 even half-lattice internal spinors,
// i.e. flat arrays of n = 12*Vh double2 chunks, one complex number per chunk.  Reductions are deterministic
// (grid_sum_last_n).  Scalars that feed later kernels stay on the device.
#include <math.h>

#include "cola_device.cuh"

namespace cola {

namespace {

constexpr int EB = 256;
constexpr int E_MAX_BLOCKS = 148 * 8;

inline unsigned eig_grid(size_t n)
{
    size_t b = (n + EB - 1) / EB;
    return (unsigned)(b < (size_t)E_MAX_BLOCKS ? b : (size_t)E_MAX_BLOCKS);
}

// out2[0..1] = <a, b> = sum conj(a) b
__global__ void __launch_bounds__(EB) eig_cdot_kernel(const double2 *a, const double2 *b, size_t n, ReduceWs red, unsigned *counter, double *out2)
{
    double v[2] = {0.0, 0.0};
    for (size_t k = (size_t)blockIdx.x * EB + threadIdx.x; k < n; k += (size_t)gridDim.x * EB) {
        const double2 x = a[k], y = b[k];
        v[0] += x.x * y.x + x.y * y.y;
        v[1] += x.x * y.y - x.y * y.x;
    }
    double tot[2];
    if (grid_sum_last_n<2>(v, red, counter, tot)) {
        out2[0] = tot[0];
        out2[1] = tot[1];
    }
}

// w += scale * c v with the complex c = (coef2[0], coef2[1]) read from device memory (scale = -1: Gram-Schmidt step)
__global__ void __launch_bounds__(EB) eig_caxpy_kernel(double2 *w, const double2 *v, size_t n, const double *coef2, double scale)
{
    const double cr = -scale * coef2[0], ci = -scale * coef2[1];
    for (size_t k = (size_t)blockIdx.x * EB + threadIdx.x; k < n; k += (size_t)gridDim.x * EB) {
        const double2 x = v[k];
        double2 y = w[k];
        y.x -= cr * x.x - ci * x.y;
        y.y -= cr * x.y + ci * x.x;
        w[k] = y;
    }
}

// out = in / sqrt(norm2[0])   (norm2 = <in, in> from eig_cdot_kernel)
__global__ void __launch_bounds__(EB) eig_normalise_kernel(double2 *out, const double2 *in, size_t n, const double *norm2)
{
    const double s = 1.0 / sqrt(norm2[0]);
    for (size_t k = (size_t)blockIdx.x * EB + threadIdx.x; k < n; k += (size_t)gridDim.x * EB) {
        const double2 x = in[k];
        out[k] = make_double2(s * x.x, s * x.y);
    }
}

// out = a*x + b*y + c*z with real a, b, c (y, z may be nullptr when their coefficient is 0)
__global__ void __launch_bounds__(EB) eig_lincomb_kernel(double2 *out, double a, const double2 *x, double b, const double2 *y, double c, const double2 *z, size_t n)
{
    for (size_t k = (size_t)blockIdx.x * EB + threadIdx.x; k < n; k += (size_t)gridDim.x * EB) {
        const double2 xv = x[k];
        double2 r = make_double2(a * xv.x, a * xv.y);
        if (y) {
            const double2 yv = y[k];
            r.x += b * yv.x;
            r.y += b * yv.y;
        }
        if (z) {
            const double2 zv = z[k];
            r.x += c * zv.x;
            r.y += c * zv.y;
        }
        out[k] = r;
    }
}

// Rotation of the basis at a restart: out[q] = sum_j V[j] Y[j][q], j < m, q < kq (real Y, m <= 64).  One thread per
// chunk: reads the m chunks once and forms kq outputs; `out` must not overlap V.  Y (m x kq, row-major) sits in global
// memory and is read through the constant cache path.
__global__ void __launch_bounds__(EB) eig_rotate_kernel(double2 *out, size_t out_stride, const double2 *V, size_t v_stride, int m, int kq, const double *Y, size_t n)
{
    for (size_t k = (size_t)blockIdx.x * EB + threadIdx.x; k < n; k += (size_t)gridDim.x * EB) {
        for (int q0 = 0; q0 < kq; q0 += 8) {
            double2 acc[8];
#pragma unroll
            for (int q = 0; q < 8; q++) acc[q] = make_double2(0.0, 0.0);
            for (int j = 0; j < m; j++) {
                const double2 x = V[(size_t)j * v_stride + k];
#pragma unroll
                for (int q = 0; q < 8; q++) {
                    if (q0 + q < kq) {
                        const double y = __ldg(Y + (size_t)j * kq + q0 + q);
                        acc[q].x += y * x.x;
                        acc[q].y += y * x.y;
                    }
                }
            }
#pragma unroll
            for (int q = 0; q < 8; q++)
                if (q0 + q < kq) out[(size_t)(q0 + q) * out_stride + k] = acc[q];
        }
    }
}

// deterministic pseudo-random start vector: a counter-based hash of (seed, real index) mapped to (-1, 1)
__global__ void __launch_bounds__(EB) eig_start_kernel(double2 *v, size_t n, unsigned long long seed)
{
    for (size_t k = (size_t)blockIdx.x * EB + threadIdx.x; k < n; k += (size_t)gridDim.x * EB) {
        double r[2];
#pragma unroll
        for (int c = 0; c < 2; c++) {
            unsigned long long z = seed + 0x9e3779b97f4a7c15ull * (2 * k + c + 1);
            z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull;
            z = (z ^ (z >> 27)) * 0x94d049bb133111ebull;
            z ^= z >> 31;
            r[c] = (double)(z >> 11) * (2.0 / 9007199254740992.0) - 1.0;
        }
        v[k] = make_double2(r[0], r[1]);
    }
}

}  // namespace

cudaError_t launch_eig_cdot(const void *a, const void *b, size_t n_sites, const ReduceWs &red, unsigned *counter, double *out2, cudaStream_t s)
{
    const size_t n = 12 * n_sites;
    eig_cdot_kernel<<<eig_grid(n), EB, 0, s>>>((const double2 *)a, (const double2 *)b, n, red, counter, out2);
    return cudaGetLastError();
}

cudaError_t launch_eig_caxpy(void *w, const void *v, size_t n_sites, const double *coef2, double scale, cudaStream_t s)
{
    const size_t n = 12 * n_sites;
    eig_caxpy_kernel<<<eig_grid(n), EB, 0, s>>>((double2 *)w, (const double2 *)v, n, coef2, scale);
    return cudaGetLastError();
}

cudaError_t launch_eig_normalise(void *out, const void *in, size_t n_sites, const double *norm2, cudaStream_t s)
{
    const size_t n = 12 * n_sites;
    eig_normalise_kernel<<<eig_grid(n), EB, 0, s>>>((double2 *)out, (const double2 *)in, n, norm2);
    return cudaGetLastError();
}

cudaError_t launch_eig_lincomb(void *out, double a, const void *x, double b, const void *y, double c, const void *z, size_t n_sites, cudaStream_t s)
{
    const size_t n = 12 * n_sites;
    eig_lincomb_kernel<<<eig_grid(n), EB, 0, s>>>((double2 *)out, a, (const double2 *)x, b, (const double2 *)y, c, (const double2 *)z, n);
    return cudaGetLastError();
}

cudaError_t launch_eig_rotate(void *out, const void *V, size_t vec_bytes, int m, int kq, const double *Y_dev, size_t n_sites, cudaStream_t s)
{
    const size_t n = 12 * n_sites;
    eig_rotate_kernel<<<eig_grid(n), EB, 0, s>>>((double2 *)out, vec_bytes / 16, (const double2 *)V, vec_bytes / 16, m, kq, Y_dev, n);
    return cudaGetLastError();
}

cudaError_t launch_eig_start(void *v, size_t n_sites, unsigned long long seed, cudaStream_t s)
{
    const size_t n = 12 * n_sites;
    eig_start_kernel<<<eig_grid(n), EB, 0, s>>>((double2 *)v, n, seed);
    return cudaGetLastError();
}

// Eigen-decomposition of the real symmetric m x m matrix A (row-major, destroyed) by cyclic Jacobi rotations (host):
// eigenvalues in w (ascending), eigenvectors as the COLUMNS of Q (row-major m x m).  m <= 64 here, a few dozen sweeps.
void jacobi_eigh(int m, double *A, double *w, double *Q)
{
    for (int i = 0; i < m; i++)
        for (int j = 0; j < m; j++) Q[i * m + j] = i == j ? 1.0 : 0.0;
    for (int sweep = 0; sweep < 100; sweep++) {
        double off = 0.0, diag = 0.0;
        for (int i = 0; i < m; i++) {
            diag += A[i * m + i] * A[i * m + i];
            for (int j = i + 1; j < m; j++) off += A[i * m + j] * A[i * m + j];
        }
        if (off <= 1e-30 * (diag + off)) break;
        for (int p = 0; p < m - 1; p++)
            for (int q = p + 1; q < m; q++) {
                const double apq = A[p * m + q];
                if (apq == 0.0) continue;
                const double theta = (A[q * m + q] - A[p * m + p]) / (2.0 * apq);
                const double t = (theta >= 0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                const double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
                for (int k = 0; k < m; k++) {   // columns p, q of A
                    const double akp = A[k * m + p], akq = A[k * m + q];
                    A[k * m + p] = c * akp - s * akq;
                    A[k * m + q] = s * akp + c * akq;
                }
                for (int k = 0; k < m; k++) {   // rows p, q of A
                    const double apk = A[p * m + k], aqk = A[q * m + k];
                    A[p * m + k] = c * apk - s * aqk;
                    A[q * m + k] = s * apk + c * aqk;
                }
                for (int k = 0; k < m; k++) {
                    const double qkp = Q[k * m + p], qkq = Q[k * m + q];
                    Q[k * m + p] = c * qkp - s * qkq;
                    Q[k * m + q] = s * qkp + c * qkq;
                }
            }
    }
    for (int i = 0; i < m; i++) w[i] = A[i * m + i];
    for (int i = 0; i < m - 1; i++) {   // selection sort, ascending, columns of Q follow
        int lo = i;
        for (int j = i + 1; j < m; j++)
            if (w[j] < w[lo]) lo = j;
        if (lo != i) {
            const double tw = w[i]; w[i] = w[lo]; w[lo] = tw;
            for (int k = 0; k < m; k++) {
                const double tq = Q[k * m + i]; Q[k * m + i] = Q[k * m + lo]; Q[k * m + lo] = tq;
            }
        }
    }
}

}  // namespace cola
