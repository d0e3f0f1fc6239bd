// linalg.cu -- spinor linear algebra on internal-layout half fields (
// PAPER.md:108-120, Fig. 7: "Copy spinor field", "g5 application", "g5 mulc add assign", inner products
// and norms).  Readings C22/C23: <a,b> = sum conj(a) b, sums in fp64; "g5 mulc add assign"
// is out += c gamma5 in.
//
// A half field is NV planes of Vh 16-byte vectors (hr_internal.h); every vector holds whole complex
// numbers, and gamma5 = diag(1,1,-1,-1) is +1 on the first NV/2 planes and -1 on the rest, so all of
// these are flat streaming kernels over nvec = NV*Vh vectors: 128-bit loads/stores, four independent
// vectors in flight per thread, grid = a multiple of the SM count.
// Reductions are ONE kernel (grid_reduce, hr_internal.h) instead of the paper's site-wise kernel followed
// by a cub reduction: the field is read once and nothing but per-CTA partials is written.
#include "hr_internal.h"

namespace hr {

template <typename Real> struct Vec16;
template <> struct Vec16<double> { using type = double2; };
template <> struct Vec16<float> { using type = float4; };

// a * b for the complex numbers packed in one 16-byte vector; a = (ar, ai) broadcast
__device__ __forceinline__ double2 cmul(double ar, double ai, double2 b) { return make_double2(ar * b.x - ai * b.y, ar * b.y + ai * b.x); }
__device__ __forceinline__ float4 cmul(float ar, float ai, float4 b)
{
    return make_float4(ar * b.x - ai * b.y, ar * b.y + ai * b.x, ar * b.z - ai * b.w, ar * b.w + ai * b.z);
}
__device__ __forceinline__ double2 vadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float4 vadd(float4 a, float4 b) { return make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w); }
__device__ __forceinline__ void dot_acc(double &re, double &im, double2 a, double2 b)
{
    re = fma(a.x, b.x, fma(a.y, b.y, re));
    im = fma(a.x, b.y, fma(-a.y, b.x, im));
}
__device__ __forceinline__ void dot_acc(double &re, double &im, float4 a, float4 b)
{
    // the products of one vector in fp32 (exact to 2^-24 each), the running sums in fp64 (reading C22)
    re += (double)(a.x * b.x + a.y * b.y) + (double)(a.z * b.z + a.w * b.w);
    im += (double)(a.x * b.y - a.y * b.x) + (double)(a.z * b.w - a.w * b.z);
}

constexpr int LIN_THREADS = 256;
constexpr int LIN_UNROLL = 4;

// out = ca * G(x) + cb * y
template <typename Real, bool G5, bool HAS_Y>
__global__ void __launch_bounds__(LIN_THREADS) lincomb_kernel(typename Vec16<Real>::type *out, const typename Vec16<Real>::type *x,
                                                              const typename Vec16<Real>::type *y, Real car, Real cai, Real cbr,
                                                              Real cbi, size_t nvec, size_t half)
{
    using V = typename Vec16<Real>::type;
    const size_t base = (size_t)blockIdx.x * (LIN_THREADS * LIN_UNROLL) + threadIdx.x;
    V xv[LIN_UNROLL], yv[LIN_UNROLL];
#pragma unroll
    for (int u = 0; u < LIN_UNROLL; ++u) {
        const size_t i = base + (size_t)u * LIN_THREADS;
        if (i < nvec) {
            xv[u] = x[i];
            if constexpr (HAS_Y) yv[u] = y[i];
        }
    }
#pragma unroll
    for (int u = 0; u < LIN_UNROLL; ++u) {
        const size_t i = base + (size_t)u * LIN_THREADS;
        if (i < nvec) {
            const Real sg = (G5 && i >= half) ? (Real)-1 : (Real)1;
            V r = cmul(sg * car, sg * cai, xv[u]);
            if constexpr (HAS_Y) r = vadd(r, cmul(cbr, cbi, yv[u]));
            out[i] = r;
        }
    }
}

// v[0] + i v[1] = <x, y>; SAME: y == x, one read
template <typename Real, bool SAME>
__global__ void __launch_bounds__(LIN_THREADS) dot_kernel(const typename Vec16<Real>::type *x, const typename Vec16<Real>::type *y,
                                                          size_t nvec, double *partial, unsigned *ticket, double *result)
{
    using V = typename Vec16<Real>::type;
    double v[2] = { 0.0, 0.0 };
    const size_t stride = (size_t)gridDim.x * (LIN_THREADS * LIN_UNROLL);
    for (size_t b0 = (size_t)blockIdx.x * (LIN_THREADS * LIN_UNROLL); b0 < nvec; b0 += stride) {
        V xv[LIN_UNROLL], yv[LIN_UNROLL];
#pragma unroll
        for (int u = 0; u < LIN_UNROLL; ++u) {
            const size_t i = b0 + threadIdx.x + (size_t)u * LIN_THREADS;
            if (i < nvec) {
                xv[u] = x[i];
                if constexpr (!SAME) yv[u] = y[i];
            }
        }
#pragma unroll
        for (int u = 0; u < LIN_UNROLL; ++u) {
            const size_t i = b0 + threadIdx.x + (size_t)u * LIN_THREADS;
            if (i < nvec) dot_acc(v[0], v[1], xv[u], SAME ? xv[u] : yv[u]);
        }
    }
    if (grid_reduce<2>(v, partial, ticket)) {
        result[0] = v[0];
        result[1] = SAME ? 0.0 : v[1];
    }
}

// ---- precision conversion of half fields in the internal layout (mixed-precision solver) -----------------------
// fp32 vector v' of site s holds the reals 4v'..4v'+3, i.e. the fp64 vectors 2v' and 2v'+1 of the same site.
__global__ void __launch_bounds__(LIN_THREADS) cvt_down_kernel(float4 *out, const double2 *in, double scale, size_t vh, size_t nvec32)
{
    const size_t i = (size_t)blockIdx.x * LIN_THREADS + threadIdx.x; // = v' * vh + s
    if (i >= nvec32) return;
    const size_t v = i / vh, s = i - v * vh;
    const double2 a = in[(2 * v) * vh + s], b = in[(2 * v + 1) * vh + s];
    out[i] = make_float4((float)(scale * a.x), (float)(scale * a.y), (float)(scale * b.x), (float)(scale * b.y));
}
// x64 += scale * (double) e32
__global__ void __launch_bounds__(LIN_THREADS) cvt_up_axpy_kernel(double2 *x, const float4 *e, double scale, size_t vh, size_t nvec32)
{
    const size_t i = (size_t)blockIdx.x * LIN_THREADS + threadIdx.x;
    if (i >= nvec32) return;
    const size_t v = i / vh, s = i - v * vh;
    const float4 ev = e[i];
    double2 a = x[(2 * v) * vh + s], b = x[(2 * v + 1) * vh + s];
    a.x = fma(scale, (double)ev.x, a.x); a.y = fma(scale, (double)ev.y, a.y);
    b.x = fma(scale, (double)ev.z, b.x); b.y = fma(scale, (double)ev.w, b.y);
    x[(2 * v) * vh + s] = a;
    x[(2 * v + 1) * vh + s] = b;
}

static inline size_t field_nvec(const hr_ctx *c, hr_prec prec) { return (size_t)c->Vh * 8 * c->d * prec_bytes(prec) / 16; }

// CTAs of a grid-stride reduction: enough to fill the machine, never more than the work
unsigned reduce_grid(size_t nvec)
{
    const size_t need = (nvec + LIN_THREADS * LIN_UNROLL - 1) / (LIN_THREADS * LIN_UNROLL);
    const size_t cap = 148 * 8;
    return (unsigned)(need < cap ? (need ? need : 1) : cap);
}

static hr_status check_launch(const char *what)
{
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) {
        set_error("%s launch failed: %s", what, cudaGetErrorString(e));
        return HR_ECUDA;
    }
    return HR_OK;
}

template <typename Real>
static hr_status lincomb_t(void *out, const double ca[2], int g5, const void *x, const double cb[2], const void *y, size_t nvec,
                           cudaStream_t st)
{
    using V = typename Vec16<Real>::type;
    const unsigned grid = (unsigned)((nvec + LIN_THREADS * LIN_UNROLL - 1) / (LIN_THREADS * LIN_UNROLL));
    const Real car = (Real)ca[0], cai = (Real)ca[1], cbr = y ? (Real)cb[0] : 0, cbi = y ? (Real)cb[1] : 0;
#define GO(G5, HY) lincomb_kernel<Real, G5, HY><<<grid, LIN_THREADS, 0, st>>>((V *)out, (const V *)x, (const V *)y, car, cai, cbr, cbi, nvec, nvec / 2)
    if (g5) { if (y) GO(true, true); else GO(true, false); }
    else    { if (y) GO(false, true); else GO(false, false); }
#undef GO
    return check_launch("lincomb_kernel");
}

hr_status launch_cvt(const hr_ctx *c, bool down, void *dst, const void *src, double scale, cudaStream_t st)
{
    const size_t nvec32 = (size_t)c->Vh * 8 * c->d * 4 / 16;
    const unsigned grid = (unsigned)((nvec32 + LIN_THREADS - 1) / LIN_THREADS);
    if (down) cvt_down_kernel<<<grid, LIN_THREADS, 0, st>>>((float4 *)dst, (const double2 *)src, scale, (size_t)c->Vh, nvec32);
    else cvt_up_axpy_kernel<<<grid, LIN_THREADS, 0, st>>>((double2 *)dst, (const float4 *)src, scale, (size_t)c->Vh, nvec32);
    return check_launch(down ? "cvt_down_kernel" : "cvt_up_axpy_kernel");
}

hr_status launch_lincomb(const hr_ctx *c, hr_prec prec, void *out, const double ca[2], int g5, const void *x, const double cb[2],
                         const void *y, cudaStream_t st)
{
    const size_t nvec = field_nvec(c, prec);
    return prec == HR_F64 ? lincomb_t<double>(out, ca, g5, x, cb, y, nvec, st) : lincomb_t<float>(out, ca, g5, x, cb, y, nvec, st);
}

template <typename Real>
static hr_status dot_t(const void *x, const void *y, size_t nvec, const RedScratch &rs, double *result, cudaStream_t st)
{
    using V = typename Vec16<Real>::type;
    const unsigned grid = reduce_grid(nvec);
    if (x == y) dot_kernel<Real, true><<<grid, LIN_THREADS, 0, st>>>((const V *)x, (const V *)y, nvec, rs.partial, rs.ticket, result);
    else dot_kernel<Real, false><<<grid, LIN_THREADS, 0, st>>>((const V *)x, (const V *)y, nvec, rs.partial, rs.ticket, result);
    return check_launch("dot_kernel");
}

hr_status launch_dot(const hr_ctx *c, hr_prec prec, const void *x, const void *y, const RedScratch &rs, double *result_dev,
                     cudaStream_t st)
{
    const size_t nvec = field_nvec(c, prec);
    return prec == HR_F64 ? dot_t<double>(x, y, nvec, rs, result_dev, st) : dot_t<float>(x, y, nvec, rs, result_dev, st);
}

// ---- fused vector updates of the gamma5-QMR (hr_qmr_dhat; real coefficients) -----------------------------------------
__device__ __forceinline__ double2 vscale(double a, double2 b) { return make_double2(a * b.x, a * b.y); }
__device__ __forceinline__ float4 vscale(float a, float4 b) { return make_float4(a * b.x, a * b.y, a * b.z, a * b.w); }
__device__ __forceinline__ double vnorm2(double2 a) { return a.x * a.x + a.y * a.y; }
__device__ __forceinline__ double vnorm2(float4 a) { return (double)(a.x * a.x + a.y * a.y) + (double)(a.z * a.z + a.w * a.w); }

// Lanczos step: w <- gamma5 w - alpha v - beta vp;  qs->red[0..1] = (|w_upper|^2, |w_lower|^2) of the new w   (3 reads, 1 write)
template <typename Real>
__global__ void __launch_bounds__(LIN_THREADS) qmr_lanczos_kernel(typename Vec16<Real>::type *w, const typename Vec16<Real>::type *v,
                                                                  const typename Vec16<Real>::type *vp, QmrState *qs,
                                                                  size_t nvec, size_t half, double *partial, unsigned *ticket)
{
    if (qs->stop != 0) return;
    const Real alpha = (Real)qs->alpha, beta = (Real)qs->beta;
    double r[2] = { 0.0, 0.0 };
    const size_t stride = (size_t)gridDim.x * LIN_THREADS;
    for (size_t i = (size_t)blockIdx.x * LIN_THREADS + threadIdx.x; i < nvec; i += stride) {
        const bool lower = i >= half;
        auto t = vadd(vscale(lower ? (Real)-1 : (Real)1, w[i]), vscale(-alpha, v[i]));
        if (beta != (Real)0) t = vadd(t, vscale(-beta, vp[i]));
        w[i] = t;
        r[lower ? 1 : 0] += vnorm2(t);
    }
    if (grid_reduce<2>(r, partial, ticket)) { qs->red[0] = r[0]; qs->red[1] = r[1]; }
}

// direction, solution and next Lanczos vector:  p2 <- (v - eps p1 - theta p2) / zeta;  x += ceta p2;  vp <- w / rho
// (5 reads, 3 writes)
template <typename Real>
__global__ void __launch_bounds__(LIN_THREADS) qmr_update_kernel(typename Vec16<Real>::type *p2, const typename Vec16<Real>::type *p1,
                                                                 const typename Vec16<Real>::type *v, typename Vec16<Real>::type *x,
                                                                 typename Vec16<Real>::type *vp, const typename Vec16<Real>::type *w,
                                                                 const QmrState *qs, size_t nvec)
{
    if (qs->do_update == 0) return;
    const size_t i = (size_t)blockIdx.x * LIN_THREADS + threadIdx.x;
    if (i >= nvec) return;
    const Real izeta = (Real)qs->izeta, eps = (Real)qs->eps, theta = (Real)qs->theta, ceta = (Real)qs->ceta, irho = (Real)qs->irho;
    const auto p = vscale(izeta, vadd(v[i], vadd(vscale(-eps, p1[i]), vscale(-theta, p2[i]))));
    p2[i] = p;
    x[i] = vadd(x[i], vscale(ceta, p));
    vp[i] = vscale(irho, w[i]);
}

// the scalar recurrences of reading C33 (oracle/solver.py::qmr_j, same order), one thread
__global__ void qmr_init_kernel(QmrState *qs, double bnorm, double delta0, double tol, int maxiter)
{
    qs->c1 = 1.0; qs->s1 = 0.0; qs->c2 = 1.0; qs->s2 = 0.0;
    qs->eta = bnorm; qs->rho = bnorm; qs->delta_prev = 1.0; qs->delta = delta0; qs->bnorm = bnorm; qs->tol = tol;
    qs->k = 0; qs->maxiter = maxiter; qs->do_update = 0;
    qs->stop = maxiter == 0 ? 4 : (delta0 == 0.0 ? 2 : 0);
    double *hist = reinterpret_cast<double *>(qs + 1);
    hist[0] = 1.0;
}
// after the Dhat launches: alpha_k = (v_k, Dhat v_k)_J / delta_k, beta_k = rho_k delta_k / delta_{k-1}
__global__ void qmr_scal_a_kernel(QmrState *qs)
{
    if (qs->stop != 0) { qs->do_update = 0; return; }
    qs->alpha = qs->red[5] / qs->delta;
    qs->beta = qs->k > 0 ? qs->rho * qs->delta / qs->delta_prev : 0.0;
}
// after the Lanczos kernel: rho_{k+1}, the two old rotations applied to the new column, the new rotation, eta
__global__ void qmr_scal_b_kernel(QmrState *qs)
{
    if (qs->stop != 0) { qs->do_update = 0; return; }
    const double up = qs->red[0], lo = qs->red[1];
    const double rho_next = sqrt(up + lo);
    const double theta = qs->s2 * qs->beta, t = qs->c2 * qs->beta;
    const double eps = qs->c1 * t + qs->s1 * qs->alpha, zt = -qs->s1 * t + qs->c1 * qs->alpha;
    const double zeta = sqrt(zt * zt + rho_next * rho_next);
    if (zeta == 0.0) { qs->stop = 2; qs->do_update = 0; return; }
    const double c = zt / zeta, s = rho_next / zeta;
    qs->izeta = 1.0 / zeta; qs->eps = eps; qs->theta = theta; qs->ceta = c * qs->eta;
    qs->irho = rho_next > 0.0 ? 1.0 / rho_next : 0.0;
    qs->do_update = 1;
    qs->eta = -s * qs->eta;
    const int k = ++qs->k;
    double *hist = reinterpret_cast<double *>(qs + 1);
    hist[k] = fabs(qs->eta) / qs->bnorm;
    qs->c2 = qs->c1; qs->s2 = qs->s1; qs->c1 = c; qs->s1 = s;
    if (rho_next == 0.0) { qs->stop = 3; return; }
    qs->delta_prev = qs->delta;
    qs->delta = (up - lo) / (up + lo);
    qs->rho = rho_next;
    if (fabs(qs->eta) <= qs->tol * qs->bnorm) qs->stop = 1;
    else if (k >= qs->maxiter) qs->stop = 4;
    else if (qs->delta == 0.0) qs->stop = 2;
}
// the host found the true residual above tol after a stop = 1: go on (or end at maxiter / at a breakdown)
__global__ void qmr_resume_kernel(QmrState *qs)
{
    qs->do_update = 0;
    qs->stop = qs->k >= qs->maxiter ? 4 : (qs->delta == 0.0 ? 2 : 0);
}

static hr_status check_small(const char *what)
{
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { set_error("%s launch failed: %s", what, cudaGetErrorString(e)); return HR_ECUDA; }
    return HR_OK;
}
hr_status launch_qmr_init(QmrState *qs, double bnorm, double delta0, double tol, int maxiter, cudaStream_t st)
{
    qmr_init_kernel<<<1, 1, 0, st>>>(qs, bnorm, delta0, tol, maxiter);
    return check_small("qmr_init_kernel");
}
hr_status launch_qmr_scal_a(QmrState *qs, cudaStream_t st) { qmr_scal_a_kernel<<<1, 1, 0, st>>>(qs); return check_small("qmr_scal_a_kernel"); }
hr_status launch_qmr_scal_b(QmrState *qs, cudaStream_t st) { qmr_scal_b_kernel<<<1, 1, 0, st>>>(qs); return check_small("qmr_scal_b_kernel"); }
hr_status launch_qmr_resume(QmrState *qs, cudaStream_t st) { qmr_resume_kernel<<<1, 1, 0, st>>>(qs); return check_small("qmr_resume_kernel"); }

template <typename Real>
static hr_status qmr_lanczos_t(void *w, const void *v, const void *vp, QmrState *qs, size_t nvec, const RedScratch &rs, cudaStream_t st)
{
    using V = typename Vec16<Real>::type;
    qmr_lanczos_kernel<Real><<<reduce_grid(nvec), LIN_THREADS, 0, st>>>((V *)w, (const V *)v, (const V *)vp, qs, nvec, nvec / 2, rs.partial, rs.ticket);
    return check_launch("qmr_lanczos_kernel");
}
template <typename Real>
static hr_status qmr_update_t(void *p2, const void *p1, const void *v, void *x, void *vp, const void *w, const QmrState *qs, size_t nvec,
                              cudaStream_t st)
{
    using V = typename Vec16<Real>::type;
    const unsigned grid = (unsigned)((nvec + LIN_THREADS - 1) / LIN_THREADS);
    qmr_update_kernel<Real><<<grid, LIN_THREADS, 0, st>>>((V *)p2, (const V *)p1, (const V *)v, (V *)x, (V *)vp, (const V *)w, qs, nvec);
    return check_launch("qmr_update_kernel");
}

hr_status launch_qmr_lanczos(const hr_ctx *c, hr_prec prec, void *w, const void *v, const void *vp, QmrState *qs, const RedScratch &rs,
                             cudaStream_t st)
{
    const size_t nvec = field_nvec(c, prec);
    return prec == HR_F64 ? qmr_lanczos_t<double>(w, v, vp, qs, nvec, rs, st) : qmr_lanczos_t<float>(w, v, vp, qs, nvec, rs, st);
}

hr_status launch_qmr_update(const hr_ctx *c, hr_prec prec, void *p2, const void *p1, const void *v, void *x, void *vp, const void *w,
                            const QmrState *qs, cudaStream_t st)
{
    const size_t nvec = field_nvec(c, prec);
    return prec == HR_F64 ? qmr_update_t<double>(p2, p1, v, x, vp, w, qs, nvec, st) : qmr_update_t<float>(p2, p1, v, x, vp, w, qs, nvec, st);
}

// <x, y> over the vectors [first, first + nvec) of the two fields (the upper / lower spin halves of a field are the first
// and second half of its vectors: gamma5 is a sign pattern on them)
hr_status launch_dot_range(const hr_ctx *c, hr_prec prec, const void *x, const void *y, size_t first, size_t nvec,
                           const RedScratch &rs, double *result_dev, cudaStream_t st)
{
    (void)c;
    const char *xp = (const char *)x + first * 16, *yp = (const char *)y + first * 16;
    return prec == HR_F64 ? dot_t<double>(xp, yp, nvec, rs, result_dev, st) : dot_t<float>(xp, yp, nvec, rs, result_dev, st);
}

} // namespace hr
