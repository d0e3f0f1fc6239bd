// dot_noalloc.cu -- hr_spinor_dot_noalloc: the inner product of two half fields (hr_spinor_dot, linalg.cu)
// for callers that may not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// hr_spinor_dot keeps its per-CTA partial sums and its ticket in a scratch buffer that the context cudaMalloc's on first use
// (get_red_scratch).  Here the same one-pass reduction (grid_reduce, hr_internal.h) runs on a FILE-SCOPE device array:
//
//   * g_dot_scratch is 256 + 16 * kNaMaxCtas bytes = 33024 bytes, resident on every GPU that loads libhr.so until the process
//     exits: [0, 256) the ticket (one unsigned), then 2 doubles per CTA;
//   * in HOST code the name g_dot_scratch is a host-side stand-in for the symbol, not a device address: a kernel given it would
//     fault (or, where the GPU can reach host memory, silently use the wrong memory).  The device address is obtained once per
//     device, with that device current, by cudaGetSymbolAddress below, and THAT pointer is what the kernel receives;
//   * the entry point calls no cudaMalloc / cudaFree / allocating library routine: cudaSetDevice, cudaGetSymbolAddress (first
//     call per device only), cudaMemsetAsync on the ticket, one kernel launch;
//   * every call on a device shares the array, which keeps the previous call's partial sums: the ticket -- the only word that
//     must start at zero -- is cleared on the caller's stream before each launch (the last CTA also wraps it back to zero, but a
//     launch that was aborted would leave it behind), the partials are overwritten before they are read.  Two calls that can
//     OVERLAP on the GPU (different streams with no dependency between them, or two host threads) RACE on the array and
//     return garbage: order them on one stream or with events.
//
// Limits: fields of at most kNaMaxVec = 2^28 16-byte vectors (4 GiB per half field) and grids of at most kNaMaxCtas CTAs;
// larger problems are rejected with HR_EUNSUPPORTED before anything is launched.  `result` must be DEVICE memory.
#include <mutex>

#include "hr_internal.h"

constexpr unsigned kNaMaxCtas = 2048;               // partial-sum slots; reduce_grid() never asks for more than 148 * 8
constexpr size_t kNaMaxVec = (size_t)1 << 28;       // 16-byte vectors per field
constexpr int kNaHeader = 32;                       // doubles reserved for the ticket (256 bytes)
constexpr int NA_THREADS = 256, NA_UNROLL = 4;      // the geometry of linalg.cu's dot_kernel: same order of summation

// the scratch: 33024 bytes on every device that loads the library.  Host code may only hand this name to cudaGetSymbolAddress.
static __device__ __align__(256) double g_dot_scratch[kNaHeader + 2 * kNaMaxCtas];

namespace hr {
unsigned reduce_grid(size_t nvec); // linalg.cu: the grid hr_spinor_dot uses
namespace {

template <typename Real> struct NaVec;
template <> struct NaVec<double> { using type = double2; };
template <> struct NaVec<float> { using type = float4; };

__device__ __forceinline__ void na_acc(double &re, double &im, double2 a, double2 b)
{
    re = fma(a.x, b.x, fma(a.y, b.y, re));
    im = fma(a.x, b.y, fma(-a.y, b.x, im));
}
__device__ __forceinline__ void na_acc(double &re, double &im, float4 a, float4 b)
{
    // products of one vector in fp32, running sums in fp64 (reading C22), as in linalg.cu
    re += (double)(a.x * b.x + a.y * b.y) + (double)(a.z * b.z + a.w * b.w);
    im += (double)(a.x * b.y - a.y * b.x) + (double)(a.z * b.w - a.w * b.z);
}

// result[0] + i result[1] = <x, y> = sum conj(x) y; scratch = the DEVICE address of g_dot_scratch
template <typename Real, bool SAME>
__global__ void __launch_bounds__(NA_THREADS) dot_noalloc_kernel(const typename NaVec<Real>::type *x, const typename NaVec<Real>::type *y,
                                                                 size_t nvec, double *scratch, double *result)
{
    using V = typename NaVec<Real>::type;
    double v[2] = { 0.0, 0.0 };
    const size_t stride = (size_t)gridDim.x * (NA_THREADS * NA_UNROLL);
    for (size_t b0 = (size_t)blockIdx.x * (NA_THREADS * NA_UNROLL); b0 < nvec; b0 += stride) {
        V xv[NA_UNROLL], yv[NA_UNROLL];
#pragma unroll
        for (int u = 0; u < NA_UNROLL; ++u) {
            const size_t i = b0 + threadIdx.x + (size_t)u * NA_THREADS;
            if (i < nvec) {
                xv[u] = x[i];
                if constexpr (!SAME) yv[u] = y[i];
            }
        }
#pragma unroll
        for (int u = 0; u < NA_UNROLL; ++u) {
            const size_t i = b0 + threadIdx.x + (size_t)u * NA_THREADS;
            if (i < nvec) na_acc(v[0], v[1], xv[u], SAME ? xv[u] : yv[u]);
        }
    }
    if (grid_reduce<2>(v, scratch + kNaHeader, reinterpret_cast<unsigned *>(scratch))) {
        result[0] = v[0];
        result[1] = SAME ? 0.0 : v[1];
    }
}

// device address of g_dot_scratch on the CURRENT device `dev`; looked up once per device
hr_status scratch_address(int dev, double **out)
{
    static std::mutex mu;
    static double *addr[64] = {};
    if (dev < 0 || dev >= 64) { set_error("hr_spinor_dot_noalloc: device ordinal %d out of range", dev); return HR_EUNSUPPORTED; }
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        double *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void **)&p, g_dot_scratch);
        if (e != cudaSuccess || !p) {
            set_error("hr_spinor_dot_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            cudaGetLastError();
            return HR_ECUDA;
        }
        addr[dev] = p;
    }
    *out = addr[dev];
    return HR_OK;
}

} // namespace
} // namespace hr

using namespace hr;

size_t hr_spinor_dot_noalloc_max_bytes(void) { return kNaMaxVec * 16; }

hr_status hr_spinor_dot_noalloc(hr_ctx *ctx, hr_prec prec, const void *x, const void *y, double *result_dev, void *stream)
{
    if (!ctx || !x || !y || !result_dev || (prec != HR_F64 && prec != HR_F32)) { set_error("hr_spinor_dot_noalloc: bad argument"); return HR_EINVAL; }
    if (((uintptr_t)x & 15) || ((uintptr_t)y & 15) || ((uintptr_t)result_dev & 7)) {
        set_error("hr_spinor_dot_noalloc: fields must be 16-byte aligned, the result 8-byte aligned");
        return HR_EINVAL;
    }
    const size_t nvec = (size_t)ctx->Vh * 8 * ctx->d * prec_bytes(prec) / 16;
    if (nvec > kNaMaxVec) {
        set_error("hr_spinor_dot_noalloc: a half field of %zu bytes exceeds the limit of %zu bytes of the allocation-free path "
                  "(use hr_spinor_dot)", nvec * 16, kNaMaxVec * 16);
        return HR_EUNSUPPORTED;
    }
    const unsigned grid = reduce_grid(nvec);
    if (grid > kNaMaxCtas) {
        set_error("hr_spinor_dot_noalloc: %u CTAs exceed the %u partial-sum slots of the static scratch", grid, kNaMaxCtas);
        return HR_EUNSUPPORTED;
    }
    hr_status rc = use_device(ctx);
    if (rc != HR_OK) return rc;
    bool dev = false;
    rc = pointer_on_device(result_dev, &dev);
    if (rc != HR_OK) return rc;
    if (!dev) { set_error("hr_spinor_dot_noalloc: `result_dev` must be device memory (no synchronisation is made)"); return HR_EINVAL; }
    double *scratch = nullptr;
    rc = scratch_address(ctx->device, &scratch);
    if (rc != HR_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaMemsetAsync(scratch, 0, kNaHeader * sizeof(double), st);   // the ticket starts at zero
    if (e != cudaSuccess) { set_error("hr_spinor_dot_noalloc: cudaMemsetAsync: %s", cudaGetErrorString(e)); return HR_ECUDA; }
    if (prec == HR_F64) {
        if (x == y) dot_noalloc_kernel<double, true><<<grid, NA_THREADS, 0, st>>>((const double2 *)x, (const double2 *)y, nvec, scratch, result_dev);
        else dot_noalloc_kernel<double, false><<<grid, NA_THREADS, 0, st>>>((const double2 *)x, (const double2 *)y, nvec, scratch, result_dev);
    } else {
        if (x == y) dot_noalloc_kernel<float, true><<<grid, NA_THREADS, 0, st>>>((const float4 *)x, (const float4 *)y, nvec, scratch, result_dev);
        else dot_noalloc_kernel<float, false><<<grid, NA_THREADS, 0, st>>>((const float4 *)x, (const float4 *)y, nvec, scratch, result_dev);
    }
    count_launch();
    e = cudaPeekAtLastError();
    if (e != cudaSuccess) { set_error("hr_spinor_dot_noalloc: kernel launch failed: %s", cudaGetErrorString(e)); return HR_ECUDA; }
    return HR_OK;
}
