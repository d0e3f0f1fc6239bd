// bicgstab.cu -- vector updates of the stabilised bi-conjugate gradient with DEVICE-RESIDENT complex scalars
// ("stabilized Bi-Conjugate Gradient [11, 19]"; reading C29 of DESIGN.md: textbook BiCGstab on Dhat
// itself, x0 = 0, shadow residual rhat = b, stop when |r_k|^2 <= tol^2 |b|^2 after a full iteration).
//
// One iteration:  bi_update_p   p = r + beta (p - omega v),  beta = (rho/rho_old)(alpha/omega)        3R 1W
//                 v = Dhat p                                   (2 Dphi launches)
//                 dot           <rhat, v>                                                             2R
//                 bi_update_s   alpha = rho / <rhat, v>;  s = r - alpha v                             2R 1W
//                 t = Dhat s                                   (2 Dphi launches; the second reduces |t|^2 and <s, t>)
//                 bi_update_xr  omega = <t, s> / |t|^2;  x += alpha p + omega s;  r = s - omega t;
//                               rho' = <rhat, r>, |r|^2, k -> k+1, convergence test                   5R 2W
// rho, alpha, omega, the counter and the stop flag live in BiState on the device: the host enqueues batches of
// iterations and reads the state once per batch; after `done` every kernel of the batch returns at once.
#include "hr_internal.h"

namespace hr {

unsigned reduce_grid(size_t nvec); // linalg.cu

struct BiState {
    double bb, tol2;
    double rho[2], rho_old[2], alpha[2], omega[2];
    double rhat_v[2];  // <rhat, v>, written by the dot kernel
    double tt_st[3];   // |t|^2, Re <s,t>, Im <s,t>, written by the fused Dphi reduction
    double rr;
    int iter, maxiter, done, pad;
    // rr history (maxiter + 1 doubles) follows
};
size_t bicgstab_state_bytes(int maxiter) { return (sizeof(BiState) + ((size_t)maxiter + 2) * sizeof(double) + 255) & ~(size_t)255; }
double *bicgstab_rhat_v(void *state) { return ((BiState *)state)->rhat_v; }
double *bicgstab_tt_st(void *state) { return ((BiState *)state)->tt_st; }
const int *bicgstab_done(void *state) { return &((BiState *)state)->done; }
void bicgstab_unpack(const void *host_copy, int *iter, int *done, double *bb) {
    const BiState *s = (const BiState *)host_copy;
    *iter = s->iter; *done = s->done; *bb = s->bb;
}
size_t bicgstab_header_bytes() { return sizeof(BiState); }

template <typename Real> struct B16;
template <> struct B16<double> { using type = double2; };
template <> struct B16<float> { using type = float4; };

struct cplx { double re, im; };
__device__ __forceinline__ cplx cdiv(cplx a, cplx b) { const double d = b.re * b.re + b.im * b.im; return { (a.re * b.re + a.im * b.im) / d, (a.im * b.re - a.re * b.im) / d }; }
__device__ __forceinline__ cplx cmulc(cplx a, cplx b) { return { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re }; }

// y + c x for the complex numbers packed in a vector
__device__ __forceinline__ double2 caxpy(double cr, double ci, double2 x, double2 y) { return make_double2(y.x + cr * x.x - ci * x.y, y.y + cr * x.y + ci * x.x); }
__device__ __forceinline__ float4 caxpy(float cr, float ci, float4 x, float4 y)
{
    return make_float4(y.x + cr * x.x - ci * x.y, y.y + cr * x.y + ci * x.x, y.z + cr * x.z - ci * x.w, y.w + cr * x.w + ci * x.z);
}
__device__ __forceinline__ double sq(double2 a) { return fma(a.x, a.x, a.y * a.y); }
__device__ __forceinline__ double sq(float4 a) { return (double)(a.x * a.x + a.y * a.y) + (double)(a.z * a.z + a.w * a.w); }
__device__ __forceinline__ void cdot(double &re, double &im, double2 a, double2 b) { re = fma(a.x, b.x, fma(a.y, b.y, re)); im = fma(a.x, b.y, fma(-a.y, b.x, im)); }
__device__ __forceinline__ void cdot(double &re, double &im, float4 a, float4 b)
{
    re += (double)(a.x * b.x + a.y * b.y) + (double)(a.z * b.z + a.w * b.w);
    im += (double)(a.x * b.y - a.y * b.x) + (double)(a.z * b.w - a.w * b.z);
}
__device__ __forceinline__ double2 zero_of(double2) { return make_double2(0, 0); }
__device__ __forceinline__ float4 zero_of(float4) { return make_float4(0, 0, 0, 0); }

constexpr int BI_THREADS = 256;
__device__ __forceinline__ double *bi_hist(BiState *s) { return (double *)(s + 1); }

template <typename Real>
__global__ void __launch_bounds__(BI_THREADS) bi_init_kernel(BiState *st, double tol, int maxiter, typename B16<Real>::type *x,
                                                             typename B16<Real>::type *r, typename B16<Real>::type *rhat,
                                                             typename B16<Real>::type *p, typename B16<Real>::type *v,
                                                             const typename B16<Real>::type *b, size_t nvec, double *partial,
                                                             unsigned *ticket)
{
    double s[1] = { 0.0 };
    for (size_t i = (size_t)blockIdx.x * BI_THREADS + threadIdx.x; i < nvec; i += (size_t)gridDim.x * BI_THREADS) {
        const auto bv = b[i];
        s[0] += sq(bv);
        r[i] = bv; rhat[i] = bv;
        x[i] = zero_of(bv); p[i] = zero_of(bv); v[i] = zero_of(bv);
    }
    if (grid_reduce<1>(s, partial, ticket)) {
        st->bb = s[0]; st->tol2 = tol * tol; st->rr = s[0];
        st->rho[0] = s[0]; st->rho[1] = 0;                       // <rhat, r> = |b|^2
        st->rho_old[0] = 1; st->rho_old[1] = 0; st->alpha[0] = 1; st->alpha[1] = 0; st->omega[0] = 1; st->omega[1] = 0;
        st->iter = 0; st->maxiter = maxiter;
        bi_hist(st)[0] = s[0];
        st->done = (maxiter <= 0 || !(s[0] > tol * tol * s[0])) ? 1 : 0;
    }
}

template <typename Real>
__global__ void __launch_bounds__(BI_THREADS) bi_update_p_kernel(const BiState *st, typename B16<Real>::type *p,
                                                                 const typename B16<Real>::type *r, const typename B16<Real>::type *v, size_t nvec)
{
    if (st->done) return;
    const cplx rho = { st->rho[0], st->rho[1] }, rho_old = { st->rho_old[0], st->rho_old[1] };
    const cplx alpha = { st->alpha[0], st->alpha[1] }, omega = { st->omega[0], st->omega[1] };
    const cplx beta = cmulc(cdiv(rho, rho_old), cdiv(alpha, omega));
    const size_t i = (size_t)blockIdx.x * BI_THREADS + threadIdx.x;
    if (i >= nvec) return;
    const auto w = caxpy((Real)-omega.re, (Real)-omega.im, v[i], p[i]);  // p - omega v
    p[i] = caxpy((Real)beta.re, (Real)beta.im, w, r[i]);                 // r + beta (.)
}

template <typename Real>
__global__ void __launch_bounds__(BI_THREADS) bi_update_s_kernel(BiState *st, typename B16<Real>::type *s, const typename B16<Real>::type *r,
                                                                 const typename B16<Real>::type *v, size_t nvec)
{
    if (st->done) return;
    const cplx alpha = cdiv({ st->rho[0], st->rho[1] }, { st->rhat_v[0], st->rhat_v[1] });
    const size_t i = (size_t)blockIdx.x * BI_THREADS + threadIdx.x;
    if (i == 0) { st->alpha[0] = alpha.re; st->alpha[1] = alpha.im; }   // read again only by later kernels
    if (i >= nvec) return;
    s[i] = caxpy((Real)-alpha.re, (Real)-alpha.im, v[i], r[i]);
}

template <typename Real>
__global__ void __launch_bounds__(BI_THREADS) bi_update_xr_kernel(BiState *st, typename B16<Real>::type *x, typename B16<Real>::type *r,
                                                                  const typename B16<Real>::type *p, const typename B16<Real>::type *s,
                                                                  const typename B16<Real>::type *t, const typename B16<Real>::type *rhat,
                                                                  size_t nvec, double *partial, unsigned *ticket)
{
    if (st->done) return;
    const cplx alpha = { st->alpha[0], st->alpha[1] };
    // omega = <t, s> / <t, t> = conj(<s, t>) / |t|^2
    const cplx omega = { st->tt_st[1] / st->tt_st[0], -st->tt_st[2] / st->tt_st[0] };
    const int k = st->iter;
    double acc[3] = { 0.0, 0.0, 0.0 }; // |r|^2, Re <rhat, r>, Im <rhat, r>
    for (size_t i = (size_t)blockIdx.x * BI_THREADS + threadIdx.x; i < nvec; i += (size_t)gridDim.x * BI_THREADS) {
        const auto sv = s[i];
        auto xv = caxpy((Real)alpha.re, (Real)alpha.im, p[i], x[i]);
        xv = caxpy((Real)omega.re, (Real)omega.im, sv, xv);
        x[i] = xv;
        const auto rv = caxpy((Real)-omega.re, (Real)-omega.im, t[i], sv);
        r[i] = rv;
        acc[0] += sq(rv);
        cdot(acc[1], acc[2], rhat[i], rv);
    }
    if (grid_reduce<3>(acc, partial, ticket)) {
        st->omega[0] = omega.re; st->omega[1] = omega.im;
        st->rho_old[0] = st->rho[0]; st->rho_old[1] = st->rho[1];
        st->rho[0] = acc[1]; st->rho[1] = acc[2];
        st->rr = acc[0];
        bi_hist(st)[k + 1] = acc[0];
        st->iter = k + 1;
        if (!(acc[0] > st->tol2 * st->bb) || k + 1 >= st->maxiter) st->done = 1;
    }
}

static inline size_t field_nvec(const hr_ctx *c, hr_prec prec) { return (size_t)c->Vh * 8 * c->d * prec_bytes(prec) / 16; }
static hr_status launched(const char *what)
{
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { set_error("%s launch failed: %s", what, cudaGetErrorString(e)); return HR_ECUDA; }
    return HR_OK;
}

#define BI_DISPATCH(KERN, GRID, ...)                                                                                      \
    if (prec == HR_F64) { using V = double2; KERN<double><<<GRID, BI_THREADS, 0, st>>>(__VA_ARGS__); }                   \
    else { using V = float4; KERN<float><<<GRID, BI_THREADS, 0, st>>>(__VA_ARGS__); }

hr_status launch_bi_init(const hr_ctx *c, hr_prec prec, void *state, double tol, int maxiter, void *x, void *r, void *rhat, void *p,
                         void *v, const void *b, const RedScratch &rs, cudaStream_t st)
{
    const size_t nvec = field_nvec(c, prec);
    BI_DISPATCH(bi_init_kernel, reduce_grid(nvec), (BiState *)state, tol, maxiter, (V *)x, (V *)r, (V *)rhat, (V *)p, (V *)v, (const V *)b, nvec, rs.partial, rs.ticket)
    return launched("bi_init_kernel");
}
hr_status launch_bi_update_p(const hr_ctx *c, hr_prec prec, const void *state, void *p, const void *r, const void *v, cudaStream_t st)
{
    const size_t nvec = field_nvec(c, prec);
    const unsigned grid = (unsigned)((nvec + BI_THREADS - 1) / BI_THREADS);
    BI_DISPATCH(bi_update_p_kernel, grid, (const BiState *)state, (V *)p, (const V *)r, (const V *)v, nvec)
    return launched("bi_update_p_kernel");
}
hr_status launch_bi_update_s(const hr_ctx *c, hr_prec prec, void *state, void *s, const void *r, const void *v, cudaStream_t st)
{
    const size_t nvec = field_nvec(c, prec);
    const unsigned grid = (unsigned)((nvec + BI_THREADS - 1) / BI_THREADS);
    BI_DISPATCH(bi_update_s_kernel, grid, (BiState *)state, (V *)s, (const V *)r, (const V *)v, nvec)
    return launched("bi_update_s_kernel");
}
hr_status launch_bi_update_xr(const hr_ctx *c, hr_prec prec, void *state, void *x, void *r, const void *p, const void *s, const void *t,
                              const void *rhat, const RedScratch &rs, cudaStream_t st)
{
    const size_t nvec = field_nvec(c, prec);
    BI_DISPATCH(bi_update_xr_kernel, reduce_grid(nvec), (BiState *)state, (V *)x, (V *)r, (const V *)p, (const V *)s, (const V *)t, (const V *)rhat, nvec, rs.partial, rs.ticket)
    return launched("bi_update_xr_kernel");
}

} // namespace hr
