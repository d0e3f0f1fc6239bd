// represent.cu -- the link map U -> U^R, one thread per link.
//
//   FUND  R = U                                           (reading C19: copy + precision conversion)
//   ADJ   R_ab = 2 tr(T_a U T_b U^dagger), T = lambda/2   (BASELINE.json:configs[2]; real, reading C7)
//         lambda in the nested generalised Gell-Mann order (reading C6): for m = 1..N-1:
//         { for i < m: S_im, A_im }, D_m.
//   SYM / ASYM  R_(ij),(kl) = n_ij n_kl (U_ik U_jl +- U_il U_jk), pairs lexicographic with i <= j
//         (i < j), n = 1/sqrt2 on a diagonal pair                      (configs[3], reading C8)
//
// The adjoint is evaluated without any generator table: with M = U lambda_b U^dagger (Hermitian),
//   1/2 tr(S_im M) = Re M_im,   1/2 tr(A_im M) = -Im M_im,   1/2 tr(D_m M) = c_m/2 (sum_{k<m} M_kk - m M_mm),
// and M itself is a sum of one or two outer products of columns of U.  Everything is unrolled on the
// compile-time N, so only the needed entries of M are ever formed.
// Memory-bound stream: reads F bytes, writes L bytes per link, both fully coalesced 128-bit planes.
#include "hr_internal.h"

namespace hr {

template <typename R> struct C2 { R re, im; };
template <typename R> __device__ __forceinline__ C2<R> cmul(C2<R> a, C2<R> b) { return { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re }; }
template <typename R> __device__ __forceinline__ C2<R> cmulc(C2<R> a, C2<R> b) /* a * conj(b) */ { return { a.re * b.re + a.im * b.im, a.im * b.re - a.re * b.im }; }

template <int N, typename R> __device__ __forceinline__ C2<R> el(const R (&u)[2 * N * N], int r, int c) { return { u[2 * (r * N + c)], u[2 * (r * N + c) + 1] }; }

// column b of the adjoint matrix from the needed entries of the Hermitian M = U lambda_b U^dagger.
// MF(r, c) returns M_rc.
template <int N, typename R, typename MF> __device__ __forceinline__ void adj_column(R *out, int b, MF M)
{
    constexpr int D = N * N - 1;
    int a = 0;
#pragma unroll
    for (int m = 1; m < N; ++m) {
#pragma unroll
        for (int i = 0; i < m; ++i) {
            const C2<R> e = M(i, m);
            out[(a++) * D + b] = e.re;
            out[(a++) * D + b] = -e.im;
        }
        R s = 0;
#pragma unroll
        for (int k = 0; k < m; ++k) s += M(k, k).re;
        s -= (R)m * M(m, m).re;
        // c_m / 2 = sqrt(2/(m(m+1))) / 2 = 1/sqrt(2 m (m+1))
        out[(a++) * D + b] = s * (R)(1.0 / sqrt(2.0 * m * (m + 1.0)));
    }
}

template <int N, typename R> __device__ __forceinline__ void rep_adjoint(const R (&u)[2 * N * N], R (&out)[(N * N - 1) * (N * N - 1)])
{
    int b = 0;
#pragma unroll
    for (int n = 1; n < N; ++n) {
#pragma unroll
        for (int j = 0; j < n; ++j) {
            // lambda_b = S_jn: M_rc = U_rj conj(U_cn) + U_rn conj(U_cj)
            adj_column<N, R>(out, b++, [&](int r, int c) {
                const C2<R> p = cmulc(el<N>(u, r, j), el<N>(u, c, n)), q = cmulc(el<N>(u, r, n), el<N>(u, c, j));
                return C2<R>{ p.re + q.re, p.im + q.im };
            });
            // lambda_b = A_jn (-i at (j,n), +i at (n,j)): M_rc = i (U_rn conj(U_cj) - U_rj conj(U_cn))
            adj_column<N, R>(out, b++, [&](int r, int c) {
                const C2<R> p = cmulc(el<N>(u, r, j), el<N>(u, c, n)), q = cmulc(el<N>(u, r, n), el<N>(u, c, j));
                return C2<R>{ -(q.im - p.im), q.re - p.re };
            });
        }
        // lambda_b = D_n = c_n diag(1,..,1,-n,0,..): M_rc = c_n (sum_{k<n} U_rk conj(U_ck) - n U_rn conj(U_cn))
        const R cn = (R)sqrt(2.0 / (n * (n + 1.0)));
        adj_column<N, R>(out, b++, [&](int r, int c) {
            C2<R> s = { 0, 0 };
#pragma unroll
            for (int k = 0; k < n; ++k) { const C2<R> p = cmulc(el<N>(u, r, k), el<N>(u, c, k)); s.re += p.re; s.im += p.im; }
            const C2<R> p = cmulc(el<N>(u, r, n), el<N>(u, c, n));
            return C2<R>{ cn * (s.re - (R)n * p.re), cn * (s.im - (R)n * p.im) };
        });
    }
}

// SIGN = +1 symmetric (pairs i <= j), -1 antisymmetric (pairs i < j)
template <int N, int SIGN, typename R, int D> __device__ __forceinline__ void rep_twoindex(const R (&u)[2 * N * N], R (&out)[2 * D * D])
{
    constexpr R RS2 = (R)0.70710678118654752440;
    int a = 0;
#pragma unroll
    for (int i = 0; i < N; ++i)
#pragma unroll
        for (int j = i; j < N; ++j) {
            if (SIGN < 0 && i == j) continue;
            int b = 0;
#pragma unroll
            for (int k = 0; k < N; ++k)
#pragma unroll
                for (int l = k; l < N; ++l) {
                    if (SIGN < 0 && k == l) continue;
                    const C2<R> p = cmul(el<N>(u, i, k), el<N>(u, j, l)), q = cmul(el<N>(u, i, l), el<N>(u, j, k));
                    const R nrm = ((i == j) ? RS2 : (R)1) * ((k == l) ? RS2 : (R)1);
                    out[2 * (a * D + b)] = nrm * (p.re + (R)SIGN * q.re);
                    out[2 * (a * D + b) + 1] = nrm * (p.im + (R)SIGN * q.im);
                    ++b;
                }
            ++a;
        }
}

template <int N, int REP> struct RepGeom {
    static constexpr int D = REP == HR_REP_FUND ? N : REP == HR_REP_ADJ ? N * N - 1 : REP == HR_REP_SYM ? N * (N + 1) / 2 : N * (N - 1) / 2;
    static constexpr int NREP = REP == HR_REP_ADJ ? D * D : 2 * D * D;   // reals of the represented matrix
    // internal row stride of a real link (hr_internal.h link_ld): d_R + 1 for an odd d_R > 8, the extra entry zero
    static constexpr int LD = (REP == HR_REP_ADJ && (D & 1) && D > 8) ? D + 1 : D;
    static constexpr int NOUT = REP == HR_REP_ADJ ? D * LD : 2 * D * D;     // reals of the internal record
};

template <int N, int REP, typename RI, typename RO>
__global__ void __launch_bounds__(128) represent_kernel(const char *__restrict__ fund, char *__restrict__ repr, long vh)
{
    using G = RepGeom<N, REP>;
    constexpr int NIN = 2 * N * N;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 8 * vh) return;
    const long q = idx / vh; // record field: [parity of the base site][mu]
    const long s = idx - q * vh;
    RI u[NIN];
    load_record<LD_STREAM, NIN>(u, fund + (size_t)q * NIN * sizeof(RI) * vh, (size_t)vh, (size_t)s, 0);
    RI r[G::NREP];
    if constexpr (REP == HR_REP_FUND) {
#pragma unroll
        for (int e = 0; e < NIN; ++e) r[e] = u[e];
    } else if constexpr (REP == HR_REP_ADJ) {
        rep_adjoint<N, RI>(u, r);
    } else {
        rep_twoindex<N, REP == HR_REP_SYM ? 1 : -1, RI, G::D>(u, r);
    }
    RO o[G::NOUT];
    if constexpr (G::LD == G::D) {
#pragma unroll
        for (int e = 0; e < G::NOUT; ++e) o[e] = (RO)r[e];
    } else {
#pragma unroll
        for (int a = 0; a < G::D; ++a)
#pragma unroll
            for (int b = 0; b < G::LD; ++b) o[a * G::LD + b] = b < G::D ? (RO)r[a * G::D + b] : (RO)0;
    }
    store_record<G::NOUT>(repr + (size_t)q * G::NOUT * sizeof(RO) * vh, (size_t)vh, (size_t)s, o);
}

template <int N, int REP>
static hr_status launch_rep(hr_prec ip, const void *fund, hr_prec op, void *repr, long vh, cudaStream_t st)
{
    const int block = 128;
    const unsigned grid = (unsigned)((8 * vh + block - 1) / block);
    const char *f = (const char *)fund;
    char *r = (char *)repr;
    if (ip == HR_F64 && op == HR_F64) represent_kernel<N, REP, double, double><<<grid, block, 0, st>>>(f, r, vh);
    else if (ip == HR_F64 && op == HR_F32) represent_kernel<N, REP, double, float><<<grid, block, 0, st>>>(f, r, vh);
    else if (ip == HR_F32 && op == HR_F64) represent_kernel<N, REP, float, double><<<grid, block, 0, st>>>(f, r, vh);
    else represent_kernel<N, REP, float, float><<<grid, block, 0, st>>>(f, r, vh);
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { set_error("represent kernel launch failed: %s", cudaGetErrorString(e)); return HR_ECUDA; }
    return HR_OK;
}

// fundamental field -> its first N-1 rows (link kind LK_ROWS of dphi_kernel.cuh): a permutation copy, one thread per link
template <int N, typename Real>
__global__ void __launch_bounds__(128) compress_kernel(const char *__restrict__ fund, char *__restrict__ rows, long vh)
{
    constexpr int NIN = 2 * N * N, NOUT = 2 * N * (N - 1);
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 8 * vh) return;
    const long q = idx / vh, s = idx - q * vh;
    Real u[NIN], o[NOUT];
    load_record<LD_STREAM, NIN>(u, fund + (size_t)q * NIN * sizeof(Real) * vh, (size_t)vh, (size_t)s, 0);
#pragma unroll
    for (int e = 0; e < NOUT; ++e) o[e] = u[e];
    store_record<NOUT>(rows + (size_t)q * NOUT * sizeof(Real) * vh, (size_t)vh, (size_t)s, o);
}

hr_status launch_compress(const hr_ctx *c, hr_prec prec, void *rows, const void *fund, cudaStream_t st)
{
    const unsigned grid = (unsigned)((8 * c->Vh + 127) / 128);
    const char *f = (const char *)fund;
    char *r = (char *)rows;
    if (c->N == 2 && prec == HR_F64) compress_kernel<2, double><<<grid, 128, 0, st>>>(f, r, c->Vh);
    else if (c->N == 2) compress_kernel<2, float><<<grid, 128, 0, st>>>(f, r, c->Vh);
    else if (c->N == 3 && prec == HR_F64) compress_kernel<3, double><<<grid, 128, 0, st>>>(f, r, c->Vh);
    else if (c->N == 3) compress_kernel<3, float><<<grid, 128, 0, st>>>(f, r, c->Vh);
    else { set_error("row compression exists for SU(2) and SU(3) only"); return HR_EUNSUPPORTED; }
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { set_error("compress kernel launch failed: %s", cudaGetErrorString(e)); return HR_ECUDA; }
    return HR_OK;
}

hr_status launch_represent(const hr_ctx *c, hr_prec in_prec, const void *fund, hr_prec out_prec, void *repr, cudaStream_t st)
{
#define X(NN, RR) if (c->N == NN && c->rep == RR) return launch_rep<NN, RR>(in_prec, fund, out_prec, repr, c->Vh, st);
    X(2, HR_REP_FUND) X(2, HR_REP_ADJ) X(2, HR_REP_SYM)
    X(3, HR_REP_FUND) X(3, HR_REP_ADJ) X(3, HR_REP_SYM) X(3, HR_REP_ASYM)
    X(4, HR_REP_FUND) X(4, HR_REP_ASYM) X(4, HR_REP_SYM) X(4, HR_REP_ADJ)
#undef X
    set_error("no link-map kernel compiled for SU(%d) representation %d", c->N, c->rep);
    return HR_EUNSUPPORTED;
}

} // namespace hr
