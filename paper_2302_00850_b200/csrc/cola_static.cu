// cola_static.cu -- cola_spinor_norm2_static: the one entry point of the library that never enters a memory
// allocator, for callers that hold nothing but device pointers (see include/cola.h for who they are).
//
// It is norm2_kernel of cola_blas.cu (fp64 accumulation, warp shuffle -> block -> last block, fixed
// order) with one difference: the buffers of the grid-wide reduction -- per-block partials, per-group partials, the
// tickets that elect the "last block" -- do not come out of a workspace the caller lent to a context.  They live in
// the file-scope device array below, which the CUDA runtime places on every GPU that loads libcola.so and keeps there
// until the process exits.  Same grid, same summation order, hence the same bits as the context path.
//
// The array's name means something only in device code.  In host code it is a host-side shadow symbol: handing it to a
// kernel as if it were a pointer makes the kernel fault (or scribble over host memory where the GPU can reach it).
// The host gets the real device address from cudaGetSymbolAddress, once per device, with that device current.
#include <mutex>
#include <stdio.h>

#include "cola_device.cuh"

namespace cola {

namespace {

constexpr int SB = 256;                      // threads per block, as cola_blas.cu
constexpr unsigned SMAX_BLOCKS = 148 * 8;    // grid cap, as cola_blas.cu: the kernel strides over longer vectors
constexpr unsigned SMAX_GROUPS = 8;          // >= ceil(SMAX_BLOCKS / REDUCE_GROUP) = 5

// Layout of the static scratch (bytes from its start).  Partials and group partials are overwritten before they are
// read in every call; the tickets must be zero when a kernel starts.
constexpr size_t OFF_PARTIALS = 0;                                   // double[SMAX_BLOCKS]
constexpr size_t OFF_GPART = 9472;                                   // double[SMAX_GROUPS]
constexpr size_t OFF_TICKETS = 9728;                                 // unsigned[SMAX_GROUPS] group tickets, then 1 top-level ticket
constexpr size_t TICKET_BYTES = (SMAX_GROUPS + 1) * sizeof(unsigned);
static_assert(OFF_GPART >= OFF_PARTIALS + SMAX_BLOCKS * sizeof(double), "partials overlap the group partials");
static_assert(OFF_TICKETS >= OFF_GPART + SMAX_GROUPS * sizeof(double), "group partials overlap the tickets");
static_assert(OFF_TICKETS + TICKET_BYTES <= COLA_STATIC_SCRATCH_BYTES, "static scratch too small");
static_assert((SMAX_BLOCKS + REDUCE_GROUP - 1) / REDUCE_GROUP <= SMAX_GROUPS, "too few group slots");

// 16 KB on every GPU that loads the library, until exit.  Shared by every call in the process.
static __device__ __align__(256) unsigned char cola_static_scratch[COLA_STATIC_SCRATCH_BYTES];

__device__ __forceinline__ double sq(const float4 &v) { return (double)(v.x * v.x + v.y * v.y) + (double)(v.z * v.z + v.w * v.w); }
__device__ __forceinline__ double sq(const double2 &v) { return v.x * v.x + v.y * v.y; }

// `scratch` is the device address of cola_static_scratch as cudaGetSymbolAddress reported it to the host.
template <typename T>
__global__ void __launch_bounds__(SB) norm2_static_kernel(const typename VT<T>::V *v, size_t n, unsigned char *scratch, double *out)
{
    ReduceWs red;
    red.partials = reinterpret_cast<double *>(scratch + OFF_PARTIALS);
    red.gpart = reinterpret_cast<double *>(scratch + OFF_GPART);
    red.gticket = reinterpret_cast<unsigned *>(scratch + OFF_TICKETS);
    red.pstride = SMAX_BLOCKS;
    red.gstride = SMAX_GROUPS;
    unsigned *counter = red.gticket + SMAX_GROUPS;
    double acc = 0.0;
    for (size_t k = (size_t)blockIdx.x * SB + threadIdx.x; k < n; k += (size_t)gridDim.x * SB) acc += sq(v[k]);
    grid_sum_finalize(acc, red, counter, out);
}

// Per-device set-up state.  ptr[d] != nullptr: cudaGetSymbolAddress has run with device d current.
constexpr int MAX_DEVICES = 64;
std::mutex g_setup_lock;
unsigned char *g_scratch_ptr[MAX_DEVICES];

cola_status sfail(cola_status st, const char *what, const char *detail = "")
{
    char buf[512];
    snprintf(buf, sizeof(buf), "cola_spinor_norm2_static: %s%s", what, detail);
    set_thread_error(buf);
    return st;
}

}  // namespace

}  // namespace cola

using namespace cola;

extern "C" cola_status cola_spinor_norm2_static(int device, void *stream, cola_prec prec, const void *v_dev, size_t n_sites, double *out_dev)
{
    if (prec != COLA_F64 && prec != COLA_F32) return sfail(COLA_EINVAL, "prec must be COLA_F64 or COLA_F32");
    if (!v_dev || !out_dev) return sfail(COLA_EINVAL, "NULL vector or result pointer");
    if (n_sites == 0) return sfail(COLA_EINVAL, "n_sites = 0");
    if (n_sites > (size_t)COLA_STATIC_MAX_SITES) return sfail(COLA_EINVAL, "n_sites exceeds COLA_STATIC_MAX_SITES (2^25 sites, the 64^3x128 lattice)");
    if (device < 0 || device >= MAX_DEVICES) return sfail(COLA_EINVAL, "device ordinal outside 0..63");
    cudaStream_t s = (cudaStream_t)stream;

    int prev = -1;
    cudaError_t e = cudaGetDevice(&prev);
    if (e != cudaSuccess) return sfail(COLA_ECUDA, "cudaGetDevice: ", cudaGetErrorString(e));
    if (prev != device) {
        e = cudaSetDevice(device);
        if (e != cudaSuccess) return sfail(COLA_ECUDA, "cudaSetDevice: ", cudaGetErrorString(e));
    }
    cola_status st = COLA_OK;
    unsigned char *scratch = nullptr;
    {
        // First call on this device: ask the runtime where this device's copy of the array is.
        std::lock_guard<std::mutex> hold(g_setup_lock);
        if (!g_scratch_ptr[device]) {
            void *p = nullptr;
            e = cudaGetSymbolAddress(&p, cola_static_scratch);
            if (e != cudaSuccess || !p) st = sfail(COLA_ECUDA, "cudaGetSymbolAddress: ", e != cudaSuccess ? cudaGetErrorString(e) : "null address");
            else g_scratch_ptr[device] = static_cast<unsigned char *>(p);
        }
        scratch = g_scratch_ptr[device];
    }
    if (st == COLA_OK) {
        // The tickets count arrivals from zero and reset themselves at the end of a launch; a launch that died half
        // way would leave them dirty for everyone after it, so every call zeroes them, in stream order, before its kernel.
        e = cudaMemsetAsync(scratch + OFF_TICKETS, 0, TICKET_BYTES, s);
        if (e != cudaSuccess) st = sfail(COLA_ECUDA, "cudaMemsetAsync: ", cudaGetErrorString(e));
    }
    if (st == COLA_OK) {
        const size_t n = (prec == COLA_F64 ? 12 : 6) * n_sites;   // 16-byte chunks
        size_t b = (n + SB - 1) / SB;
        const unsigned grid = (unsigned)(b < (size_t)SMAX_BLOCKS ? b : (size_t)SMAX_BLOCKS);
        if (prec == COLA_F64) norm2_static_kernel<double><<<grid, SB, 0, s>>>((const double2 *)v_dev, n, scratch, out_dev);
        else norm2_static_kernel<float><<<grid, SB, 0, s>>>((const float4 *)v_dev, n, scratch, out_dev);
        e = cudaGetLastError();
        if (e != cudaSuccess) st = sfail(COLA_ECUDA, "kernel launch: ", cudaGetErrorString(e));
    }
    if (prev != device && prev >= 0) cudaSetDevice(prev);
    return st;
}
