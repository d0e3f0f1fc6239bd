// cg.cu -- vector updates of the conjugate gradient with DEVICE-RESIDENT scalars (SURVEY.md section 8(f)
// NEXT-1; "Conjugate Gradient"; reading C21 of DESIGN.md: textbook CG on
// A = Dhat^dagger Dhat = (gamma5 Dhat)^2, x0 = 0, recursive residual, stop when |r_k|^2 <= tol^2 |rhs|^2).
//
// One iteration is   t = Q p, Ap = Q t  (4 Dphi launches; the second one reduces pap = |Q p|^2 = <p, A p>
// in its epilogue),  cg_update_r:  r -= alpha Ap, rr[k+1] = |r|^2   (alpha = rr[k] / pap),
//                    cg_update_xp: x += alpha p,  p = r + beta p    (beta = rr[k+1] / rr[k]).
// alpha, beta, the iteration counter and the convergence flags live in CgState on the device, so the host
// enqueues iterations without ever waiting for a scalar; once `done` is set the remaining launches of a
// batch return at once.  Eight field passes of linear algebra per iteration (2R+1W, 3R+2W).
#include "hr_internal.h"

namespace hr {

unsigned reduce_grid(size_t nvec); // linalg.cu

template <typename Real> struct V16;
template <> struct V16<double> { using type = double2; };
template <> struct V16<float> { using type = float4; };

__device__ __forceinline__ double2 axpy(double a, double2 x, double2 y) { return make_double2(fma(a, x.x, y.x), fma(a, x.y, y.y)); }
__device__ __forceinline__ float4 axpy(float a, float4 x, float4 y)
{
    return make_float4(fmaf(a, x.x, y.x), fmaf(a, x.y, y.y), fmaf(a, x.z, y.z), fmaf(a, x.w, y.w));
}
__device__ __forceinline__ double sq(double2 a) { return fma(a.x, a.x, a.y * a.y); }
__device__ __forceinline__ double sq(float4 a) { return (double)(a.x * a.x + a.y * a.y) + (double)(a.z * a.z + a.w * a.w); }
__device__ __forceinline__ double2 vzero(double2) { return make_double2(0, 0); }
__device__ __forceinline__ float4 vzero(float4) { return make_float4(0, 0, 0, 0); }

constexpr int CG_THREADS = 256;
constexpr int CG_UNROLL = 4;

__device__ __forceinline__ double *cg_rr(CgState *cs) { return (double *)(cs + 1); }
__device__ __forceinline__ const double *cg_rr(const CgState *cs) { return (const double *)(cs + 1); }

// x = 0, p = r, rr[0] = bb = |r|^2, state reset
template <typename Real>
__global__ void __launch_bounds__(CG_THREADS) cg_init_kernel(CgState *cs, double tol, int maxiter, typename V16<Real>::type *x,
                                                             typename V16<Real>::type *p, const typename V16<Real>::type *r,
                                                             size_t nvec, double *partial, unsigned *ticket)
{
    using V = typename V16<Real>::type;
    double v[1] = { 0.0 };
    const size_t stride = (size_t)gridDim.x * (CG_THREADS * CG_UNROLL);
    for (size_t b0 = (size_t)blockIdx.x * (CG_THREADS * CG_UNROLL); b0 < nvec; b0 += stride) {
#pragma unroll
        for (int u = 0; u < CG_UNROLL; ++u) {
            const size_t i = b0 + threadIdx.x + (size_t)u * CG_THREADS;
            if (i < nvec) {
                const V rv = r[i];
                v[0] += sq(rv);
                p[i] = rv;
                x[i] = vzero(rv);
            }
        }
    }
    if (grid_reduce<1>(v, partial, ticket)) {
        cs->bb = v[0];
        cs->tol2 = tol * tol;
        cs->pap = 0.0;
        cs->iter = 0;
        cs->maxiter = maxiter;
        cg_rr(cs)[0] = v[0];
        const int done = (maxiter <= 0 || !(v[0] > tol * tol * v[0])) ? 1 : 0;
        cs->done = done;
        cs->frozen = done;
    }
}

// r -= alpha Ap, rr[k+1] = |r|^2, k -> k+1, convergence test
template <typename Real>
__global__ void __launch_bounds__(CG_THREADS) cg_update_r_kernel(CgState *cs, typename V16<Real>::type *r,
                                                                 const typename V16<Real>::type *Ap, size_t nvec,
                                                                 double *partial, unsigned *ticket)
{
    using V = typename V16<Real>::type;
    if (cs->done) {
        if (blockIdx.x == 0 && threadIdx.x == 0) cs->frozen = 1;
        return;
    }
    const int k = cs->iter;
    const double rrk = cg_rr(cs)[k];
    const Real malpha = (Real)(-(rrk / cs->pap));
    double v[1] = { 0.0 };
    const size_t stride = (size_t)gridDim.x * (CG_THREADS * CG_UNROLL);
    for (size_t b0 = (size_t)blockIdx.x * (CG_THREADS * CG_UNROLL); b0 < nvec; b0 += stride) {
        V rv[CG_UNROLL], av[CG_UNROLL];
#pragma unroll
        for (int u = 0; u < CG_UNROLL; ++u) {
            const size_t i = b0 + threadIdx.x + (size_t)u * CG_THREADS;
            if (i < nvec) { rv[u] = r[i]; av[u] = Ap[i]; }
        }
#pragma unroll
        for (int u = 0; u < CG_UNROLL; ++u) {
            const size_t i = b0 + threadIdx.x + (size_t)u * CG_THREADS;
            if (i < nvec) {
                const V n = axpy(malpha, av[u], rv[u]);
                v[0] += sq(n);
                r[i] = n;
            }
        }
    }
    if (grid_reduce<1>(v, partial, ticket)) {
        cg_rr(cs)[k + 1] = v[0];
        cs->iter = k + 1;
        if (!(v[0] > cs->tol2 * cs->bb) || k + 1 >= cs->maxiter) cs->done = 1;
    }
}

// x += alpha p, p = r + beta p   (of the iteration the r-update has just completed)
template <typename Real>
__global__ void __launch_bounds__(CG_THREADS) cg_update_xp_kernel(const CgState *cs, typename V16<Real>::type *x,
                                                                  typename V16<Real>::type *p, const typename V16<Real>::type *r,
                                                                  size_t nvec)
{
    using V = typename V16<Real>::type;
    if (cs->frozen) return;
    const int k1 = cs->iter; // >= 1
    const double rr0 = cg_rr(cs)[k1 - 1], rr1 = cg_rr(cs)[k1];
    const Real alpha = (Real)(rr0 / cs->pap), beta = (Real)(rr1 / rr0);
    const size_t base = (size_t)blockIdx.x * (CG_THREADS * CG_UNROLL) + threadIdx.x;
    V xv[CG_UNROLL], pv[CG_UNROLL], rv[CG_UNROLL];
#pragma unroll
    for (int u = 0; u < CG_UNROLL; ++u) {
        const size_t i = base + (size_t)u * CG_THREADS;
        if (i < nvec) { xv[u] = x[i]; pv[u] = p[i]; rv[u] = r[i]; }
    }
#pragma unroll
    for (int u = 0; u < CG_UNROLL; ++u) {
        const size_t i = base + (size_t)u * CG_THREADS;
        if (i < nvec) {
            x[i] = axpy(alpha, pv[u], xv[u]);
            p[i] = axpy(beta, pv[u], rv[u]);
        }
    }
}

static inline size_t field_nvec(const hr_ctx *c, hr_prec prec) { return (size_t)c->Vh * 8 * c->d * prec_bytes(prec) / 16; }

static hr_status launched(const char *what)
{
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) {
        set_error("%s launch failed: %s", what, cudaGetErrorString(e));
        return HR_ECUDA;
    }
    return HR_OK;
}

hr_status launch_cg_init(const hr_ctx *c, hr_prec prec, CgState *cs, double tol, int maxiter, void *x, void *p, const void *r,
                         const RedScratch &rs, cudaStream_t st)
{
    const size_t nvec = field_nvec(c, prec);
    const unsigned grid = reduce_grid(nvec);
    if (prec == HR_F64)
        cg_init_kernel<double><<<grid, CG_THREADS, 0, st>>>(cs, tol, maxiter, (double2 *)x, (double2 *)p, (const double2 *)r, nvec, rs.partial, rs.ticket);
    else
        cg_init_kernel<float><<<grid, CG_THREADS, 0, st>>>(cs, tol, maxiter, (float4 *)x, (float4 *)p, (const float4 *)r, nvec, rs.partial, rs.ticket);
    return launched("cg_init_kernel");
}

hr_status launch_cg_update_r(const hr_ctx *c, hr_prec prec, CgState *cs, void *r, const void *Ap, const RedScratch &rs, cudaStream_t st)
{
    const size_t nvec = field_nvec(c, prec);
    const unsigned grid = reduce_grid(nvec);
    if (prec == HR_F64)
        cg_update_r_kernel<double><<<grid, CG_THREADS, 0, st>>>(cs, (double2 *)r, (const double2 *)Ap, nvec, rs.partial, rs.ticket);
    else
        cg_update_r_kernel<float><<<grid, CG_THREADS, 0, st>>>(cs, (float4 *)r, (const float4 *)Ap, nvec, rs.partial, rs.ticket);
    return launched("cg_update_r_kernel");
}

hr_status launch_cg_update_xp(const hr_ctx *c, hr_prec prec, const CgState *cs, void *x, void *p, const void *r, cudaStream_t st)
{
    const size_t nvec = field_nvec(c, prec);
    const unsigned grid = (unsigned)((nvec + CG_THREADS * CG_UNROLL - 1) / (CG_THREADS * CG_UNROLL));
    if (prec == HR_F64)
        cg_update_xp_kernel<double><<<grid, CG_THREADS, 0, st>>>(cs, (double2 *)x, (double2 *)p, (const double2 *)r, nvec);
    else
        cg_update_xp_kernel<float><<<grid, CG_THREADS, 0, st>>>(cs, (float4 *)x, (float4 *)p, (const float4 *)r, nvec);
    return launched("cg_update_xp_kernel");
}

} // namespace hr
