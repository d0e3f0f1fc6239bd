// clover.cu -- SURVEY.md section 8(f) NEXT-4: the clover (Sheikholeslami-Wohlert) term ("clover [17]").
// Reading C28:
//     D_sw = D + T,   T(x) = -(c_sw/2) sum_{mu<nu} sigma_{mu nu} (x) F_{mu nu}(x),
//     F = (Q - Q^dagger)/(8i),  Q = the four counter-clockwise leaves at x from the REPRESENTED links.
// In the chiral basis of reading C1 sigma_{mu nu} is block diagonal with Pauli-matrix blocks
//     upper (spin 0,1):  s01 = sx, s02 = sy, s03 = sz, s12 = -sz, s13 = sy, s23 = -sx
//     lower (spin 2,3):  s01 = -sx, s02 = -sy, s03 = -sz, s12 = -sz, s13 = sy, s23 = -sx
// so T(x) = diag(T_up, T_dn) with  T_b = -(c_sw/2) [[C, A - iB], [A + iB, -C]]  (d_R x d_R blocks),
//     up: A = F01 - F23, B = F02 + F13, C = F03 - F12;   dn: A = -F01 - F23, B = -F02 + F13, C = -F03 - F12.
// CLOVER FIELD LAYOUT: per parity, per site one record of 2 (2 d_R)^2 reals in the plane layout of hr_internal.h:
// for each block the 2 d_R real diagonal entries, then the strict upper triangle row by row as (re, im).
//
// clover_build_kernel: one thread per site, set-up cost (once per gauge field; the Dirac operator is applied
// hundreds of times per field in a solve), written with runtime loops over d_R.
// clover_apply_kernel: out += T in, one thread per (site, chirality block), Hermitian block mat-vec unrolled on d_R;
// algorithmic bytes per site: C + 3S (clover record, in, out read, out written).
#include <type_traits>

#include "hr_internal.h"

namespace hr {

template <typename Real, int D, bool RL> struct CloverGeom {
    static constexpr int LNREAL = RL ? D * D : 2 * D * D;
    static constexpr int BLK = 4 * D * D;   // reals per packed Hermitian 2D x 2D block
    static constexpr int NREAL = 2 * BLK;
};

// one element of a link record in the plane layout of hr_internal.h (tail planes included), default caching
template <int NREAL> __device__ __forceinline__ void load_real_any(double &r, const char *base, size_t vh, size_t s, int e)
{
    constexpr int NV = NREAL / 2;
    if (NREAL % 2 == 0 || (e >> 1) < NV) r = *(const double *)(base + ((size_t)(e >> 1) * vh + s) * 16 + (size_t)(e & 1) * 8);
    else r = *(const double *)(base + (size_t)NV * 16 * vh + s * 8);
}
template <int NREAL> __device__ __forceinline__ void load_real_any(float &r, const char *base, size_t vh, size_t s, int e)
{
    constexpr int NV = NREAL / 4, TAIL = NREAL - 4 * NV;
    if (TAIL == 0 || (e >> 2) < NV) r = *(const float *)(base + ((size_t)(e >> 2) * vh + s) * 16 + (size_t)(e & 3) * 4);
    else r = *(const float *)(base + (size_t)NV * 16 * vh + s * (size_t)(TAIL * 4) + (size_t)(e - 4 * NV) * 4);
}
template <int NREAL> __device__ __forceinline__ void load_cplx_any(double &re, double &im, const char *base, size_t vh, size_t s, int e)
{
    const double2 v = *(const double2 *)(base + ((size_t)e * vh + s) * 16);
    re = v.x; im = v.y;
}
template <int NREAL> __device__ __forceinline__ void load_cplx_any(float &re, float &im, const char *base, size_t vh, size_t s, int e)
{
    constexpr int NV = NREAL / 4;
    const float2 v = (NREAL % 4 == 0 || (e >> 1) < NV) ? *(const float2 *)(base + ((size_t)(e >> 1) * vh + s) * 16 + (size_t)(e & 1) * 8)
                                                        : *(const float2 *)(base + (size_t)NV * 16 * vh + s * 8);
    re = v.x; im = v.y;
}

// complex D x D matrices as Real[2*D*D], row-major (re, im)
template <typename Real, int D, bool DA, bool DB>
__device__ __forceinline__ void cmm(Real *o, const Real *a, const Real *b) // o = op(a) op(b), op = dagger if flagged
{
    // d_R <= 4: fully unrolled, operands stay in registers; larger d_R: runtime loops over local arrays (set-up kernel)
#pragma unroll(D <= 4 ? D : 1)
    for (int i = 0; i < D; ++i)
#pragma unroll(D <= 4 ? D : 1)
        for (int j = 0; j < D; ++j) {
            Real re = 0, im = 0;
#pragma unroll(D <= 4 ? D : 1)
            for (int k = 0; k < D; ++k) {
                const int ia = DA ? 2 * (k * D + i) : 2 * (i * D + k);
                const int ib = DB ? 2 * (j * D + k) : 2 * (k * D + j);
                const Real ar = a[ia], ai = DA ? -a[ia + 1] : a[ia + 1];
                const Real br = b[ib], bi = DB ? -b[ib + 1] : b[ib + 1];
                re += ar * br - ai * bi;
                im += ar * bi + ai * br;
            }
            o[2 * (i * D + j)] = re;
            o[2 * (i * D + j) + 1] = im;
        }
}

struct CloverArgs {
    void *clover;
    const void *links;
    const void *in;
    void *out;
    int T, X, Y, Z;
    long vh;
    double csw;
};

template <typename Real, int D, bool RL>
__device__ void load_link(Real *m, const CloverArgs &a, int t, int x, int y, int z, int mu)
{
    constexpr int LNREAL = CloverGeom<Real, D, RL>::LNREAL;
    t = (t + a.T) % a.T; x = (x + a.X) % a.X; y = (y + a.Y) % a.Y; z = (z + a.Z) % a.Z;
    const int q = (t + x + y + z) & 1;
    const size_t s = (((size_t)t * a.X + x) * a.Y + y) * (a.Z / 2) + z / 2;
    const size_t LB = (size_t)LNREAL * sizeof(Real);
    const char *base = (const char *)a.links + (size_t)(q * 4 + mu) * LB * (size_t)a.vh;
    Real r[LNREAL];
    load_record<LD_DEFAULT, LNREAL>(r, base, (size_t)a.vh, s, 0);
    if constexpr (RL) {
        for (int e = 0; e < D * D; ++e) { m[2 * e] = r[e]; m[2 * e + 1] = 0; }
    } else {
        for (int e = 0; e < 2 * D * D; ++e) m[e] = r[e];
    }
}

// q += op(m1) op(m2) op(m3) op(m4)
template <typename Real, int D, bool D1, bool D2, bool D3, bool D4>
__device__ void add_leaf(Real *q, const Real *m1, const Real *m2, const Real *m3, const Real *m4)
{
    Real p[2 * D * D], r[2 * D * D];
    cmm<Real, D, D1, D2>(p, m1, m2);
    cmm<Real, D, false, D3>(r, p, m3);
    cmm<Real, D, false, D4>(p, r, m4);
    for (int e = 0; e < 2 * D * D; ++e) q[e] += p[e];
}

template <typename Real, int D, bool RL>
__global__ void __launch_bounds__(64) clover_build_kernel(const CloverArgs a)
{
    using G = CloverGeom<Real, D, RL>;
    constexpr int M = 2 * D * D;
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x; // full-lattice lexicographic index
    if (i >= 2 * a.vh) return;
    int c[4];
    {
        long r = i;
        c[3] = (int)(r % a.Z); r /= a.Z;
        c[2] = (int)(r % a.Y); r /= a.Y;
        c[1] = (int)(r % a.X);
        c[0] = (int)(r / a.X);
    }
    // coefficient matrices of sx, sy, sz in the two chirality blocks
    Real cf[2][3][M];
    for (int b = 0; b < 2; ++b)
        for (int k = 0; k < 3; ++k)
            for (int e = 0; e < M; ++e) cf[b][k][e] = 0;
    // plane (mu,nu) -> (Pauli index, sign in the upper block, sign in the lower block)
    const int pk[6] = { 0, 1, 2, 2, 1, 0 };
    const int su[6] = { 1, 1, 1, -1, 1, -1 };
    const int sd[6] = { -1, -1, -1, -1, 1, -1 };
    int plane = 0;
    for (int mu = 0; mu < 4; ++mu)
        for (int nu = mu + 1; nu < 4; ++nu, ++plane) {
            auto at = [&](int dm, int dn, int dir, Real *m) {
                int y[4] = { c[0], c[1], c[2], c[3] };
                y[mu] += dm;
                y[nu] += dn;
                load_link<Real, D, RL>(m, a, y[0], y[1], y[2], y[3], dir);
            };
            Real q[M], m1[M], m2[M], m3[M], m4[M];
            for (int e = 0; e < M; ++e) q[e] = 0;
            // U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
            at(0, 0, mu, m1); at(1, 0, nu, m2); at(0, 1, mu, m3); at(0, 0, nu, m4);
            add_leaf<Real, D, false, false, true, true>(q, m1, m2, m3, m4);
            // U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
            at(0, 0, nu, m1); at(-1, 1, mu, m2); at(-1, 0, nu, m3); at(-1, 0, mu, m4);
            add_leaf<Real, D, false, true, true, false>(q, m1, m2, m3, m4);
            // U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
            at(-1, 0, mu, m1); at(-1, -1, nu, m2); at(-1, -1, mu, m3); at(0, -1, nu, m4);
            add_leaf<Real, D, true, true, false, false>(q, m1, m2, m3, m4);
            // U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag
            at(0, -1, nu, m1); at(0, -1, mu, m2); at(1, -1, nu, m3); at(0, 0, mu, m4);
            add_leaf<Real, D, true, false, false, true>(q, m1, m2, m3, m4);
            // F = (Q - Q^dag)/(8i):  F_re = Im(Q - Q^dag)/8, F_im = -Re(Q - Q^dag)/8
            for (int r = 0; r < D; ++r)
                for (int s = 0; s < D; ++s) {
                    const Real gre = q[2 * (r * D + s)] - q[2 * (s * D + r)];
                    const Real gim = q[2 * (r * D + s) + 1] + q[2 * (s * D + r) + 1];
                    const Real fre = gim * (Real)0.125, fim = -gre * (Real)0.125;
                    cf[0][pk[plane]][2 * (r * D + s)] += su[plane] * fre;
                    cf[0][pk[plane]][2 * (r * D + s) + 1] += su[plane] * fim;
                    cf[1][pk[plane]][2 * (r * D + s)] += sd[plane] * fre;
                    cf[1][pk[plane]][2 * (r * D + s) + 1] += sd[plane] * fim;
                }
        }
    // T_b = -(c_sw/2) [[C, A - iB], [A + iB, -C]], packed: diagonal, then strict upper triangle (re, im)
    const Real k = (Real)(-0.5 * a.csw);
    Real rec[G::NREAL];
    for (int b = 0; b < 2; ++b) {
        const Real *A = cf[b][0], *B = cf[b][1], *C = cf[b][2];
        auto elem = [&](int row, int col, Real &re, Real &im) {
            const int sr = row / D, ar = row % D, sc = col / D, ac = col % D;
            const int e = 2 * (ar * D + ac);
            if (sr == 0 && sc == 0) { re = C[e]; im = C[e + 1]; }
            else if (sr == 1 && sc == 1) { re = -C[e]; im = -C[e + 1]; }
            else if (sr == 0 && sc == 1) { re = A[e] + B[e + 1]; im = A[e + 1] - B[e]; }   // A - iB
            else { re = A[e] - B[e + 1]; im = A[e + 1] + B[e]; }                           // A + iB
            re *= k; im *= k;
        };
        Real *o = rec + b * G::BLK;
        int w = 0;
        for (int d = 0; d < 2 * D; ++d) { Real re, im; elem(d, d, re, im); o[w++] = re; }
        for (int r = 0; r < 2 * D; ++r)
            for (int s = r + 1; s < 2 * D; ++s) { Real re, im; elem(r, s, re, im); o[w++] = re; o[w++] = im; }
    }
    const int qpar = (c[0] + c[1] + c[2] + c[3]) & 1;
    const size_t hs = (size_t)(i >> 1);
    char *base = (char *)a.clover + (size_t)qpar * G::NREAL * sizeof(Real) * (size_t)a.vh;
    store_record<G::NREAL>(base, (size_t)a.vh, hs, rec);
}

// ---- plane-parallel build for d_R <= 4 -----------------------------------------------------------------------------------
// One thread per (site, plane (mu, nu)): Q_{mu nu}(x) = the sum of the four plaquette leaves around x, each
// ((M1 M2) M3) M4 with the links loaded just before the product that needs them and the link shared by two consecutive
// leaves (U_nu(x), U_mu(x-mu), U_nu(x-nu)) kept in registers: 13 link loads and 12 products per thread, live state
// q + two partial products + two links.  The plane is uniform over a CTA (blockIdx.y) and a compile-time constant of the
// code path; neighbour sites come from the lexicographic index by adding a stride (the wrap is a compare, not a modulo).
// F goes to the scratch layout of clover_q_kernel, clover_pack_f_kernel finishes.  (clover_build_kernel above holds all six
// planes of a site in one thread: 252 registers and 1.5 KB of local memory in fp64, and four integer divisions per link.)
template <typename Real, int D, bool RL, int MU, int NU>
__device__ __forceinline__ void clover_plane(const CloverArgs &a, const int (&c)[4], int par, long lex, Real (&q)[2 * D * D])
{
    constexpr int M = 2 * D * D;
    constexpr int LNREAL = CloverGeom<Real, D, RL>::LNREAL;
    const size_t vh = (size_t)a.vh;
    const int ext[4] = { a.T, a.X, a.Y, a.Z };
    const long str[4] = { (long)a.X * a.Y * a.Z, (long)a.Y * a.Z, (long)a.Z, 1 };
    // displacement of the lexicographic index by +-1 in mu / nu
    const long dmu[3] = { c[MU] == 0 ? (long)(ext[MU] - 1) * str[MU] : -str[MU], 0, c[MU] == ext[MU] - 1 ? -(long)(ext[MU] - 1) * str[MU] : str[MU] };
    const long dnu[3] = { c[NU] == 0 ? (long)(ext[NU] - 1) * str[NU] : -str[NU], 0, c[NU] == ext[NU] - 1 ? -(long)(ext[NU] - 1) * str[NU] : str[NU] };
    auto link = [&](Real (&m)[M], int dm, int dn, int dir) {
        const size_t s = (size_t)((lex + dmu[dm + 1] + dnu[dn + 1]) >> 1);
        const int qy = par ^ ((dm + dn) & 1);
        const char *base = (const char *)a.links + (size_t)(qy * 4 + dir) * LNREAL * sizeof(Real) * vh;
        if constexpr (RL) {
            Real r[LNREAL];
            load_record<LD_DEFAULT, LNREAL>(r, base, vh, s, 0);
#pragma unroll
            for (int e = 0; e < D * D; ++e) { m[2 * e] = r[e]; m[2 * e + 1] = 0; }
        } else {
            load_record<LD_DEFAULT, LNREAL>(m, base, vh, s, 0);
        }
    };
    Real p[M], r[M], u[M], v[M];
#pragma unroll
    for (int e = 0; e < M; ++e) q[e] = 0;
    // U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
    link(u, 0, 0, MU); link(v, 1, 0, NU);
    cmm<Real, D, false, false>(p, u, v);
    link(u, 0, 1, MU);
    cmm<Real, D, false, true>(r, p, u);
    link(v, 0, 0, NU);                                           // U_nu(x): also the first factor of the next leaf
    cmm<Real, D, false, true>(p, r, v);
#pragma unroll
    for (int e = 0; e < M; ++e) q[e] += p[e];
    // U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
    link(u, -1, 1, MU);
    cmm<Real, D, false, true>(p, v, u);
    link(u, -1, 0, NU);
    cmm<Real, D, false, true>(r, p, u);
    link(v, -1, 0, MU);                                          // U_mu(x-mu): first factor of the next leaf
    cmm<Real, D, false, false>(p, r, v);
#pragma unroll
    for (int e = 0; e < M; ++e) q[e] += p[e];
    // U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
    link(u, -1, -1, NU);
    cmm<Real, D, true, true>(p, v, u);
    link(u, -1, -1, MU);
    cmm<Real, D, false, false>(r, p, u);
    link(v, 0, -1, NU);                                          // U_nu(x-nu): first factor of the next leaf
    cmm<Real, D, false, false>(p, r, v);
#pragma unroll
    for (int e = 0; e < M; ++e) q[e] += p[e];
    // U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag
    link(u, 0, -1, MU);
    cmm<Real, D, true, false>(p, v, u);
    link(u, 1, -1, NU);
    cmm<Real, D, false, false>(r, p, u);
    link(v, 0, 0, MU);
    cmm<Real, D, false, true>(p, r, v);
#pragma unroll
    for (int e = 0; e < M; ++e) q[e] += p[e];
}

template <typename Real, int D, bool RL>
__global__ void __launch_bounds__(64) clover_plane_kernel(const CloverArgs a, Real *scratch, long first, long n)
{
    constexpr int M = 2 * D * D;
    const long loc = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (loc >= n) return;
    const long idx = first + loc;                                  // even-odd site index: [parity][half index]
    const int par = idx >= a.vh ? 1 : 0;
    int c[4];
    long lex;
    {
        long r = idx - (long)par * a.vh;
        const int Zh = a.Z / 2;
        const int zh = (int)(r % Zh); r /= Zh;
        c[2] = (int)(r % a.Y); r /= a.Y;
        c[1] = (int)(r % a.X);
        c[0] = (int)(r / a.X);
        c[3] = 2 * zh + ((c[0] + c[1] + c[2] + par) & 1);
        lex = (((long)c[0] * a.X + c[1]) * a.Y + c[2]) * a.Z + c[3];
    }
    Real q[M];
    const int plane = (int)blockIdx.y;                             // (0,1) (0,2) (0,3) (1,2) (1,3) (2,3)
    switch (plane) {
    case 0: clover_plane<Real, D, RL, 0, 1>(a, c, par, lex, q); break;
    case 1: clover_plane<Real, D, RL, 0, 2>(a, c, par, lex, q); break;
    case 2: clover_plane<Real, D, RL, 0, 3>(a, c, par, lex, q); break;
    case 3: clover_plane<Real, D, RL, 1, 2>(a, c, par, lex, q); break;
    case 4: clover_plane<Real, D, RL, 1, 3>(a, c, par, lex, q); break;
    default: clover_plane<Real, D, RL, 2, 3>(a, c, par, lex, q); break;
    }
    // F = (Q - Q^dag)/(8i):  F_re = Im(Q - Q^dag)/8, F_im = -Re(Q - Q^dag)/8  (as clover_build_kernel / clover_pack_vec_kernel)
    // scratch: [plane][real index 2 (row D + col) + re/im][site of the chunk]
#pragma unroll
    for (int r = 0; r < D; ++r)
#pragma unroll
        for (int c2 = 0; c2 < D; ++c2) {
            const Real gre = q[2 * (r * D + c2)] - q[2 * (c2 * D + r)];
            const Real gim = q[2 * (r * D + c2) + 1] + q[2 * (c2 * D + r) + 1];
            scratch[((size_t)plane * M + 2 * (r * D + c2)) * (size_t)n + (size_t)loc] = gim * (Real)0.125;
            scratch[((size_t)plane * M + 2 * (r * D + c2) + 1) * (size_t)n + (size_t)loc] = -gre * (Real)0.125;
        }
}

// T from the six F of clover_plane_kernel, d_R <= 4: one thread per site, every index a compile-time constant (no local
// arrays); an element of T is formed from the two or four F entries it needs (coalesced loads from the scratch, which the
// plane kernel has just left in L2) and leaves through a 16-byte vector as soon as the vector is complete.
//   up: A = F01 - F23, B = F02 + F13, C = F03 - F12;   dn: A = -F01 - F23, B = -F02 + F13, C = -F03 - F12
//   T_b = -(c_sw/2) [[C, A - iB], [A + iB, -C]], packed: the 2 d_R diagonal entries, then the strict upper triangle
template <typename Real, int D, bool RL>
__global__ void __launch_bounds__(128) clover_pack_f_kernel(const CloverArgs a, const Real *scratch, long first, long n)
{
    using G = CloverGeom<Real, D, RL>;
    constexpr int M = 2 * D * D, RPV = 16 / (int)sizeof(Real);
    const long loc = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (loc >= n) return;
    const long idx = first + loc;
    const int qpar = idx >= a.vh ? 1 : 0;
    const size_t hs = (size_t)(idx - (long)qpar * a.vh), vh = (size_t)a.vh;
    char *out = (char *)a.clover + (size_t)qpar * G::NREAL * sizeof(Real) * vh + hs * 16;
    const Real k = (Real)(-0.5 * a.csw);
    auto F = [&](int plane, int e) -> Real { return scratch[((size_t)plane * M + e) * (size_t)n + (size_t)loc]; };
    // planes: 0 (0,1)  1 (0,2)  2 (0,3)  3 (1,2)  4 (1,3)  5 (2,3)
    static_assert(G::BLK % RPV == 0, "a block is a whole number of vectors");
#pragma unroll 1
    for (int b = 0; b < 2; ++b) {
        const Real sg = b ? (Real)-1 : (Real)1;                    // sign of F01, F02, F03 in the block
        char *ob = out + (size_t)(b * (G::BLK / RPV)) * vh * 16;
        Real buf[RPV];
        int w = 0;                                                 // position in the block: compile-time once unrolled
        auto put = [&](Real v) {
            buf[w % RPV] = v;
            if (++w % RPV == 0) {
                if constexpr (sizeof(Real) == 8) st16<ST_DEFAULT>(ob + (size_t)(w / RPV - 1) * vh * 16, buf[0], buf[1]);
                else st16<ST_DEFAULT>(ob + (size_t)(w / RPV - 1) * vh * 16, buf[0], buf[1], buf[2], buf[3]);
            }
        };
        auto elem = [&](int row, int col, Real &re, Real &im) {
            const int sr = row / D, ar = row % D, sc = col / D, ac = col % D;
            const int e = 2 * (ar * D + ac);
            if (sr == sc) {                                         // +-C, C = +-F03 - F12
                const Real cr = sg * F(2, e) - F(3, e), ci = sg * F(2, e + 1) - F(3, e + 1);
                re = sr ? -cr : cr; im = sr ? -ci : ci;
            } else {                                                // (0,1): A - iB,  A = +-F01 - F23, B = +-F02 + F13
                const Real Ar = sg * F(0, e) - F(5, e), Ai = sg * F(0, e + 1) - F(5, e + 1);
                const Real Br = sg * F(1, e) + F(4, e), Bi = sg * F(1, e + 1) + F(4, e + 1);
                re = Ar + Bi; im = Ai - Br;
            }
            re *= k; im *= k;
        };
#pragma unroll
        for (int d = 0; d < 2 * D; ++d) { Real re, im; elem(d, d, re, im); put(re); }
#pragma unroll
        for (int r = 0; r < 2 * D; ++r)
#pragma unroll
            for (int c2 = 0; c2 < 2 * D; ++c2)                      // rectangular bounds: the compiler unrolls them fully
                if (c2 > r) { Real re, im; elem(r, c2, re, im); put(re); put(im); }
    }
}

// ---- row-parallel build for d_R > 4 ------------------------------------------------------------------------------------
// clover_build_kernel keeps d_R x d_R matrices in thread-local arrays and is bound by local-memory traffic from d_R = 6 on
// (80 ms for the sextet at 24^3 x 48).  Here one thread owns ONE ROW of the plaquette products: row_i(M1 M2 M3 M4) =
// ((e_i^T M1) M2) M3) M4 is three vector-matrix products with the vector (d_R complex) in registers and the matrices
// streamed from the link field through L1 -- the d_R threads of a site (d_R warps of a CTA, lanes = consecutive sites:
// coalesced element loads) read the same links.  clover_q_kernel writes the rows of Q_{mu nu} (sum of the four leaves)
// of a chunk of sites to a scratch buffer; clover_pack_vec_kernel forms F = (Q - Q^dagger)/(8i) and packs T as above.
struct LeafFactor { signed char dm, dn, nu_dir, dag; };          // site offset (in mu, nu), link direction (0 mu / 1 nu), dagger
__constant__ LeafFactor kLeaf[4][4] = {
    { { 0, 0, 0, 0 }, { 1, 0, 1, 0 }, { 0, 1, 0, 1 }, { 0, 0, 1, 1 } },       // U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
    { { 0, 0, 1, 0 }, { -1, 1, 0, 1 }, { -1, 0, 1, 1 }, { -1, 0, 0, 0 } },    // U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
    { { -1, 0, 0, 1 }, { -1, -1, 1, 1 }, { -1, -1, 0, 0 }, { 0, -1, 1, 0 } }, // U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
    { { 0, -1, 1, 1 }, { 0, -1, 0, 0 }, { 1, -1, 1, 0 }, { 0, 0, 0, 1 } } };  // U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag

template <typename Real, int D, bool RL>
__global__ void __launch_bounds__(32 * D) clover_q_kernel(const CloverArgs a, Real *scratch, long first, long n)
{
    constexpr int LNREAL = CloverGeom<Real, D, RL>::LNREAL;
    const int lane = (int)threadIdx.x & 31, row = (int)threadIdx.x >> 5;
    const long loc = (long)blockIdx.x * 32 + lane;
    if (loc >= n) return;
    const long idx = first + loc;                                  // even-odd site index: [parity][half index]
    const int par = idx >= a.vh ? 1 : 0;
    int c[4];
    {
        long r = idx - (long)par * a.vh;
        const int Zh = a.Z / 2;
        const int zh = (int)(r % Zh); r /= Zh;
        c[2] = (int)(r % a.Y); r /= a.Y;
        c[1] = (int)(r % a.X);
        c[0] = (int)(r / a.X);
        c[3] = 2 * zh + ((c[0] + c[1] + c[2] + par) & 1);
    }
    const int ext[4] = { a.T, a.X, a.Y, a.Z };
    const size_t vh = (size_t)a.vh;
    int plane = 0;
    for (int mu = 0; mu < 4; ++mu)
        for (int nu = mu + 1; nu < 4; ++nu, ++plane) {
            Real q[2 * D];
#pragma unroll
            for (int j = 0; j < 2 * D; ++j) q[j] = 0;
            for (int leaf = 0; leaf < 4; ++leaf) {
                Real r[2 * D];
                for (int f = 0; f < 4; ++f) {
                    const LeafFactor lf = kLeaf[leaf][f];
                    int y[4] = { c[0], c[1], c[2], c[3] };
                    y[mu] = (y[mu] + lf.dm + ext[mu]) % ext[mu];
                    y[nu] = (y[nu] + lf.dn + ext[nu]) % ext[nu];
                    const int qy = (y[0] + y[1] + y[2] + y[3]) & 1;
                    const size_t sy = (((size_t)y[0] * a.X + y[1]) * a.Y + y[2]) * (a.Z / 2) + y[3] / 2;
                    const char *base = (const char *)a.links + (size_t)(qy * 4 + (lf.nu_dir ? nu : mu)) * LNREAL * sizeof(Real) * vh;
                    const bool dag = lf.dag != 0;
                    auto elem = [&](int k, int j, Real &re, Real &im) {       // op(M)[k][j]
                        const int e = dag ? j * D + k : k * D + j;
                        if constexpr (RL) { load_real_any<LNREAL>(re, base, vh, sy, e); im = 0; }
                        else { load_cplx_any<LNREAL>(re, im, base, vh, sy, e); if (dag) im = -im; }
                    };
                    if (f == 0) {
#pragma unroll
                        for (int j = 0; j < D; ++j) elem(row, j, r[2 * j], r[2 * j + 1]);
                    } else {
                        Real rn[2 * D];
#pragma unroll
                        for (int j = 0; j < 2 * D; ++j) rn[j] = 0;
#pragma unroll
                        for (int k = 0; k < D; ++k)
#pragma unroll
                            for (int j = 0; j < D; ++j) {
                                Real mr, mi;
                                elem(k, j, mr, mi);
                                rn[2 * j] = fma(r[2 * k], mr, fma(-r[2 * k + 1], mi, rn[2 * j]));
                                rn[2 * j + 1] = fma(r[2 * k], mi, fma(r[2 * k + 1], mr, rn[2 * j + 1]));
                            }
#pragma unroll
                        for (int j = 0; j < 2 * D; ++j) r[j] = rn[j];
                    }
                }
#pragma unroll
                for (int j = 0; j < 2 * D; ++j) q[j] += r[j];
            }
            // scratch: [plane][real index 2 (row D + j) + re/im][site of the chunk]
#pragma unroll
            for (int j = 0; j < 2 * D; ++j) scratch[((size_t)plane * 2 * D * D + (size_t)row * 2 * D + j) * (size_t)n + (size_t)loc] = q[j];
        }
}

// clover_q_kernel with the links staged through shared memory: there the d_R row-threads of a site each fetch
// all d_R^2 elements of every factor from L1 (d_R times the same matrix: 2736 element loads per thread at d_R = 6, one per four
// FMAs -- the load/store unit binds it: 3.2 ms per 77k-site chunk).  Here the CTA (32 sites x d_R rows) copies a factor's
// matrices once, d_R elements per thread, into one of two shared-memory buffers [element][site] and every row-thread reads
// its operands from there (consecutive lanes = consecutive 16-byte words: conflict-free); the copy of the next factor is
// issued before the arithmetic of this one, one barrier per factor.  Same products in the same order: same bits.
template <typename Real> struct StagedReal { Real x; static constexpr Real y = 0; };   // a real link element (adjoint representation)
template <typename Real, int D, bool RL>
__global__ void __launch_bounds__(32 * D) clover_q_staged_kernel(const CloverArgs a, Real *scratch, long first, long n)
{
    constexpr int LNREAL = CloverGeom<Real, D, RL>::LNREAL;
    using C2c = typename std::conditional<sizeof(Real) == 8, double2, float2>::type;
    using C2r = typename std::conditional<RL, StagedReal<Real>, C2c>::type;
    __shared__ C2r stg[2][D * D][32];
    const int lane = (int)threadIdx.x & 31, row = (int)threadIdx.x >> 5;
    long loc = (long)blockIdx.x * 32 + lane;
    const bool live = loc < n;
    if (!live) loc = n - 1;                                        // every thread stays for the barriers
    const long idx = first + loc;                                  // even-odd site index: [parity][half index]
    const int par = idx >= a.vh ? 1 : 0;
    int c[4];
    {
        long r = idx - (long)par * a.vh;
        const int Zh = a.Z / 2;
        const int zh = (int)(r % Zh); r /= Zh;
        c[2] = (int)(r % a.Y); r /= a.Y;
        c[1] = (int)(r % a.X);
        c[0] = (int)(r / a.X);
        c[3] = 2 * zh + ((c[0] + c[1] + c[2] + par) & 1);
    }
    const int ext[4] = { a.T, a.X, a.Y, a.Z };
    const size_t vh = (size_t)a.vh;
    // factor g = ((plane * 4 + leaf) * 4 + f), g = 0 .. 95: copy my d_R elements (row `row` of the stored matrix) into buffer g & 1
    auto stage = [&](int g) {
        const int f = g & 3, leaf = (g >> 2) & 3, plane = g >> 4;
        const int mu = plane < 3 ? 0 : plane < 5 ? 1 : 2, nu = plane < 3 ? plane + 1 : plane < 5 ? plane - 1 : 3;
        const LeafFactor lf = kLeaf[leaf][f];
        int y[4] = { c[0], c[1], c[2], c[3] };
        y[mu] = (y[mu] + lf.dm + ext[mu]) % ext[mu];
        y[nu] = (y[nu] + lf.dn + ext[nu]) % ext[nu];
        const int qy = (y[0] + y[1] + y[2] + y[3]) & 1;
        const size_t sy = (((size_t)y[0] * a.X + y[1]) * a.Y + y[2]) * (a.Z / 2) + y[3] / 2;
        const char *base = (const char *)a.links + (size_t)(qy * 4 + (lf.nu_dir ? nu : mu)) * LNREAL * sizeof(Real) * vh;
#pragma unroll
        for (int j = 0; j < D; ++j) {
            C2r v;
            if constexpr (RL) load_real_any<LNREAL>(v.x, base, vh, sy, row * D + j);
            else { Real re, im; load_cplx_any<LNREAL>(re, im, base, vh, sy, row * D + j); v.x = re; v.y = im; }
            stg[g & 1][row * D + j][lane] = v;
        }
    };
    stage(0);
    __syncthreads();
    Real q[2 * D], r[2 * D];
    for (int g = 0; g < 96; ++g) {
        const int f = g & 3, leaf = (g >> 2) & 3, plane = g >> 4;
        if (g + 1 < 96) stage(g + 1);                                  // the other buffer: free since the barrier of factor g - 1
        const bool dag = kLeaf[leaf][f].dag != 0;
        const C2r (*m)[32] = stg[g & 1];
        if (f == 0 && leaf == 0) {
#pragma unroll
            for (int j = 0; j < 2 * D; ++j) q[j] = 0;
        }
        if (f == 0) {                                                  // r = row `row` of op(M)
#pragma unroll
            for (int j = 0; j < D; ++j) {
                const C2r v = dag ? m[j * D + row][lane] : m[row * D + j][lane];
                r[2 * j] = v.x; r[2 * j + 1] = dag ? -v.y : v.y;
            }
        } else {                                                       // r = r op(M)
            Real rn[2 * D];
#pragma unroll
            for (int j = 0; j < 2 * D; ++j) rn[j] = 0;
#pragma unroll
            for (int k = 0; k < D; ++k)
#pragma unroll
                for (int j = 0; j < D; ++j) {
                    const C2r v = dag ? m[j * D + k][lane] : m[k * D + j][lane];
                    const Real mr = v.x, mi = dag ? -v.y : v.y;
                    rn[2 * j] = fma(r[2 * k], mr, fma(-r[2 * k + 1], mi, rn[2 * j]));
                    rn[2 * j + 1] = fma(r[2 * k], mi, fma(r[2 * k + 1], mr, rn[2 * j + 1]));
                }
#pragma unroll
            for (int j = 0; j < 2 * D; ++j) r[j] = rn[j];
        }
        if (f == 3) {
#pragma unroll
            for (int j = 0; j < 2 * D; ++j) q[j] += r[j];
            if (leaf == 3 && live) {
#pragma unroll
                for (int j = 0; j < 2 * D; ++j) scratch[((size_t)plane * 2 * D * D + (size_t)row * 2 * D + j) * (size_t)n + (size_t)loc] = q[j];
            }
        }
        __syncthreads();                                               // buffer g & 1 may be overwritten, buffer (g + 1) & 1 is complete
    }
}

// T from the six Q of the row-parallel kernels, any d_R: one thread per (site, 16-byte vector of the packed record) -- no
// per-thread matrices at all (its predecessor held cf[2][3][2 d_R^2] per thread in local memory: 5.8 KB of stack at d_R = 6).  A
// thread decodes which packed reals its vector holds, forms each from the F entries it needs (F = (Q - Q^dag)/(8i) on the
// fly: two Q loads per F entry, coalesced over the sites of the chunk) and stores the vector; consecutive threads are
// consecutive sites of the same vector, so loads and stores are coalesced.
template <typename Real, int D, bool RL>
__global__ void __launch_bounds__(128) clover_pack_vec_kernel(const CloverArgs a, const Real *scratch, long first, long n)
{
    using G = CloverGeom<Real, D, RL>;
    constexpr int M = 2 * D * D, N2 = 2 * D, RPV = 16 / (int)sizeof(Real), NVREC = G::NREAL / RPV, NVBLK = G::BLK / RPV;
    const long tid = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= n * NVREC) return;
    const int v = (int)(tid / n);                                  // vector of the record
    const long loc = tid - (long)v * n;
    const long idx = first + loc;
    const int qpar = idx >= a.vh ? 1 : 0;
    const size_t hs = (size_t)(idx - (long)qpar * a.vh), vh = (size_t)a.vh;
    const int b = v / NVBLK;                                       // chirality block
    const Real sg = b ? (Real)-1 : (Real)1, kk = (Real)(-0.5 * a.csw);
    auto Q = [&](int plane, int e) -> Real { return scratch[((size_t)plane * M + e) * (size_t)n + (size_t)loc]; };
    auto Fre = [&](int plane, int r, int c) -> Real { return (Q(plane, 2 * (r * D + c) + 1) + Q(plane, 2 * (c * D + r) + 1)) * (Real)0.125; };
    auto Fim = [&](int plane, int r, int c) -> Real { return -(Q(plane, 2 * (r * D + c)) - Q(plane, 2 * (c * D + r))) * (Real)0.125; };
    // planes: 0 (0,1)  1 (0,2)  2 (0,3)  3 (1,2)  4 (1,3)  5 (2,3);  up: A = F01 - F23, B = F02 + F13, C = F03 - F12, dn: F0k -> -F0k
    auto elem = [&](int row, int col, int part) -> Real {          // part 0 re, 1 im of T_b[row][col], row <= col
        const int sr = row / D, ar = row % D, sc = col / D, ac = col % D;
        Real val;
        if (sr == sc) {
            const Real c = part == 0 ? sg * Fre(2, ar, ac) - Fre(3, ar, ac) : sg * Fim(2, ar, ac) - Fim(3, ar, ac);
            val = sr ? -c : c;
        } else if (part == 0) val = (sg * Fre(0, ar, ac) - Fre(5, ar, ac)) + (sg * Fim(1, ar, ac) + Fim(4, ar, ac));   // Re(A - iB) = A_re + B_im
        else val = (sg * Fim(0, ar, ac) - Fim(5, ar, ac)) - (sg * Fre(1, ar, ac) + Fre(4, ar, ac));                    // Im(A - iB) = A_im - B_re
        return val * kk;
    };
    Real out[RPV];
#pragma unroll
    for (int i = 0; i < RPV; ++i) {
        const int w = (v - b * NVBLK) * RPV + i;                   // packed real of the block
        if (w < N2) out[i] = elem(w, w, 0);
        else {
            int u = (w - N2) >> 1, r = 0;
            while (u >= N2 - 1 - r) { u -= N2 - 1 - r; ++r; }
            out[i] = elem(r, r + 1 + u, (w - N2) & 1);
        }
    }
    char *dst = (char *)a.clover + (size_t)qpar * G::NREAL * sizeof(Real) * vh + ((size_t)v * vh + hs) * 16;
    if constexpr (sizeof(Real) == 8) st16<ST_DEFAULT>(dst, out[0], out[1]);
    else st16<ST_DEFAULT>(dst, out[0], out[1], out[2], out[3]);
}

// out += T in on one parity (clover/in/out point at that parity's half fields).  One thread per (site, chirality
// block): it holds the block's 2 d_R input and output components and STREAMS the packed Hermitian block through one
// 16-byte vector at a time (a whole d_R = 6 block is 144 reals -- preloading it spills).
// MODE: +1  out += T in;   0  out = T in (out is not read);   -1  out = T in - out
template <typename Real, int D, int MODE>
__global__ void __launch_bounds__(128) clover_apply_kernel(const CloverArgs a)
{
    constexpr int BLK = 4 * D * D, N2 = 2 * D, RPV = 16 / (int)sizeof(Real);
    constexpr int NVB = BLK / RPV;         // vectors per block record
    constexpr int NVH = 4 * D / RPV;       // vectors of two spin components of a spinor
    static_assert(BLK % RPV == 0 && (4 * D) % RPV == 0, "block and half spinor are whole vectors");
    const long tid = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const long s = tid >> 1;
    const int b = (int)(tid & 1);
    if (s >= a.vh) return;
    const size_t vh = (size_t)a.vh, pb = vh * 16;
    Real v[4 * D], w[4 * D];
    load_planes<LD_STREAM, NVH>(v, (const char *)a.in + (size_t)s * 16 + (size_t)(b * NVH) * pb, pb, 0);
    if constexpr (MODE == 0) {
#pragma unroll
        for (int e = 0; e < 4 * D; ++e) w[e] = 0;
    } else {
        load_planes<LD_STREAM, NVH>(w, (const char *)a.out + (size_t)s * 16 + (size_t)(b * NVH) * pb, pb, 0);
        if constexpr (MODE < 0) {
#pragma unroll
            for (int e = 0; e < 4 * D; ++e) w[e] = -w[e];
        }
    }
    const char *tp = (const char *)a.clover + (size_t)s * 16 + (size_t)(b * NVB) * pb;
    Real tv[RPV];
    int idx = 0; // position in the packed block; a compile-time constant at every use once the loops are unrolled
    auto next = [&]() -> Real {
        if (idx % RPV == 0) load_planes<LD_STREAM, 1>(tv, tp + (size_t)(idx / RPV) * pb, pb, 0);
        return tv[idx++ % RPV];
    };
#pragma unroll
    for (int d = 0; d < N2; ++d) {                            // diagonal entries (real)
        const Real t = next();
        w[2 * d] = fma(t, v[2 * d], w[2 * d]);
        w[2 * d + 1] = fma(t, v[2 * d + 1], w[2 * d + 1]);
    }
#pragma unroll
    for (int r = 0; r < N2; ++r)
#pragma unroll
        for (int c = r + 1; c < N2; ++c) {                    // T_rc = re + i im, T_cr = its conjugate
            const Real re = next();
            const Real im = next();
            w[2 * r] = fma(re, v[2 * c], fma(-im, v[2 * c + 1], w[2 * r]));
            w[2 * r + 1] = fma(re, v[2 * c + 1], fma(im, v[2 * c], w[2 * r + 1]));
            w[2 * c] = fma(re, v[2 * r], fma(im, v[2 * r + 1], w[2 * c]));
            w[2 * c + 1] = fma(re, v[2 * r + 1], fma(-im, v[2 * r], w[2 * c + 1]));
        }
    store_planes<ST_DEFAULT, NVH>((char *)a.out + (size_t)s * 16 + (size_t)(b * NVH) * pb, pb, w);
}

// In-place  T -> E = m [exp(T/m) - 1]  on the packed Hermitian blocks (reading C31: exponentiated clover).
// One thread per (site, chirality block): the n x n block (n = 2 d_R <= 16) is unpacked to a dense complex matrix,
// X = T / (m 2^6) is exponentiated by a 10-term Taylor series of expm1 (|X| < 0.1: remainder < 1e-22) and the result
// is squared six times in the expm1 form  e(2X) = e(X)^2 + 2 e(X)  (no cancellation against the identity), then
// packed back.  Set-up kernel: runtime loops over local arrays.
// position of (r, c), r < c, in the packed strict upper triangle (row by row) of an N x N Hermitian matrix
template <int N> __host__ __device__ constexpr int up(int r, int c) { return r * (2 * N - r - 1) / 2 + (c - r - 1); }

// A Hermitian N x N matrix in registers: N real diagonal entries and the strict upper triangle; every index compile-time.
template <int N> struct Herm {
    double d[N], re[N * (N - 1) / 2], im[N * (N - 1) / 2];
    __device__ __forceinline__ double er(int r, int c) const { return r == c ? d[r] : r < c ? re[up<N>(r, c)] : re[up<N>(c, r)]; }
    __device__ __forceinline__ double ei(int r, int c) const { return r == c ? 0.0 : r < c ? im[up<N>(r, c)] : -im[up<N>(c, r)]; }
};
// C = A B for COMMUTING Hermitian A, B (polynomials of one matrix): the product is Hermitian, only its upper triangle is formed
template <int N> __device__ __forceinline__ void herm_mul(Herm<N> &c, const Herm<N> &a, const Herm<N> &b)
{
#pragma unroll
    for (int r = 0; r < N; ++r)
#pragma unroll
        for (int cc = 0; cc < N; ++cc)
            if (cc >= r) {
                double sr = 0, si = 0;
#pragma unroll
                for (int k = 0; k < N; ++k) {
                    const double ar = a.er(r, k), ai = a.ei(r, k), br = b.er(k, cc), bi = b.ei(k, cc);
                    sr += ar * br - ai * bi;
                    if (cc > r) si += ar * bi + ai * br;
                }
                if (cc == r) c.d[r] = sr;
                else { c.re[up<N>(r, cc)] = sr; c.im[up<N>(r, cc)] = si; }
            }
}

template <typename Real, int D>
__global__ void __launch_bounds__(64) clover_exp_kernel(char *clover, long vh, double m)
{
    constexpr int N2 = 2 * D, M = 2 * N2 * N2, BLK = 4 * D * D, RPV = 16 / (int)sizeof(Real), NVB = BLK / RPV;
    const long tid = (long)blockIdx.x * blockDim.x + threadIdx.x; // over 2 parities x vh sites x 2 blocks
    if (tid >= 4 * vh) return;
    const int b = (int)(tid & 1);
    const long site = tid >> 1;                                    // 0 .. 2 vh
    const long par = site / vh, s = site - par * vh;
    char *rec = clover + (size_t)par * 2 * BLK * sizeof(Real) * (size_t)vh + (size_t)s * 16 + (size_t)(b * NVB) * (size_t)vh * 16;
    const size_t pb = (size_t)vh * 16;
    Real t[BLK];
    load_planes<LD_DEFAULT, NVB>(t, rec, pb, 0);
    if constexpr (D <= 3) {
        // d_R <= 3: the same algorithm on Hermitian matrices held in registers (X, its powers and expm1(X) are Hermitian and
        // commute): expm1(X) by Horner, s_k = (X + X s_{k+1}) / k from s_11 = 0 down to s_1, then six squarings
        constexpr int NU = N2 * (N2 - 1) / 2;
        const double sc = 1.0 / (m * 64.0);
        Herm<N2> x, e, q;
#pragma unroll
        for (int d = 0; d < N2; ++d) x.d[d] = (double)t[d] * sc;
#pragma unroll
        for (int u = 0; u < NU; ++u) { x.re[u] = (double)t[N2 + 2 * u] * sc; x.im[u] = (double)t[N2 + 2 * u + 1] * sc; }
#pragma unroll
        for (int d = 0; d < N2; ++d) e.d[d] = x.d[d] * 0.1;
#pragma unroll
        for (int u = 0; u < NU; ++u) { e.re[u] = x.re[u] * 0.1; e.im[u] = x.im[u] * 0.1; }
#pragma unroll 1
        for (int k = 9; k >= 1; --k) {
            herm_mul<N2>(q, x, e);
            const double ik = 1.0 / k;
#pragma unroll
            for (int d = 0; d < N2; ++d) e.d[d] = (x.d[d] + q.d[d]) * ik;
#pragma unroll
            for (int u = 0; u < NU; ++u) { e.re[u] = (x.re[u] + q.re[u]) * ik; e.im[u] = (x.im[u] + q.im[u]) * ik; }
        }
#pragma unroll 1
        for (int sq = 0; sq < 6; ++sq) {                               // expm1(2X) = expm1(X)^2 + 2 expm1(X)
            herm_mul<N2>(q, e, e);
#pragma unroll
            for (int d = 0; d < N2; ++d) e.d[d] = q.d[d] + 2.0 * e.d[d];
#pragma unroll
            for (int u = 0; u < NU; ++u) { e.re[u] = q.re[u] + 2.0 * e.re[u]; e.im[u] = q.im[u] + 2.0 * e.im[u]; }
        }
#pragma unroll
        for (int d = 0; d < N2; ++d) t[d] = (Real)(m * e.d[d]);
#pragma unroll
        for (int u = 0; u < NU; ++u) { t[N2 + 2 * u] = (Real)(m * e.re[u]); t[N2 + 2 * u + 1] = (Real)(m * e.im[u]); }
        store_planes<ST_DEFAULT, NVB>(rec, pb, t);
        return;
    }
    double x[M], e[M], p[M], q[M];
    const double sc = 1.0 / (m * 64.0);
    for (int i = 0; i < M; ++i) x[i] = 0;
    {
        int w = 0;
        for (int d = 0; d < N2; ++d) x[2 * (d * N2 + d)] = (double)t[w++] * sc;
        for (int r = 0; r < N2; ++r)
            for (int c = r + 1; c < N2; ++c) {
                const double re = (double)t[w++] * sc, im = (double)t[w++] * sc;
                x[2 * (r * N2 + c)] = re; x[2 * (r * N2 + c) + 1] = im;
                x[2 * (c * N2 + r)] = re; x[2 * (c * N2 + r) + 1] = -im;
            }
    }
    auto mul = [&](double *o, const double *a, const double *bb) {   // o = a bb (dense complex N2 x N2)
        for (int i = 0; i < N2; ++i)
            for (int j = 0; j < N2; ++j) {
                double re = 0, im = 0;
                for (int k = 0; k < N2; ++k) {
                    const double ar = a[2 * (i * N2 + k)], ai = a[2 * (i * N2 + k) + 1];
                    const double br = bb[2 * (k * N2 + j)], bi = bb[2 * (k * N2 + j) + 1];
                    re += ar * br - ai * bi;
                    im += ar * bi + ai * br;
                }
                o[2 * (i * N2 + j)] = re; o[2 * (i * N2 + j) + 1] = im;
            }
    };
    // e = expm1(X) = X + X^2/2! + ... + X^10/10!
    for (int i = 0; i < M; ++i) { e[i] = x[i]; p[i] = x[i]; }
    for (int k = 2; k <= 10; ++k) {
        mul(q, p, x);
        for (int i = 0; i < M; ++i) { p[i] = q[i] / k; e[i] += p[i]; }
    }
    for (int sq = 0; sq < 6; ++sq) {                                  // expm1(2X) = expm1(X)^2 + 2 expm1(X)
        mul(q, e, e);
        for (int i = 0; i < M; ++i) e[i] = q[i] + 2.0 * e[i];
    }
    {
        int w = 0;
        for (int d = 0; d < N2; ++d) t[w++] = (Real)(m * e[2 * (d * N2 + d)]);
        for (int r = 0; r < N2; ++r)
            for (int c = r + 1; c < N2; ++c) { t[w++] = (Real)(m * e[2 * (r * N2 + c)]); t[w++] = (Real)(m * e[2 * (r * N2 + c) + 1]); }
    }
    store_planes<ST_DEFAULT, NVB>(rec, pb, t);
}

// d_R >= 4: ONE WARP per block.  The thread-per-block kernel above keeps four dense n x n complex matrices (n = 2 d_R = 12: 9 KB)
// in local memory and takes 93 ms for the sextet at 24^3 x 48.  Here the three matrices of the Horner / squaring scheme
// (X, E, Q; dense, n^2 complex each) live in shared memory, the n (n + 1) / 2 upper-triangle entries of a product of two
// commuting Hermitian matrices are shared out over the 32 lanes (the lower triangle is the mirror image), and the record
// is read and written by the lanes vector by vector.  Same algorithm, same fp64 arithmetic.
#ifndef HR_CLV_EXP_PAD
#define HR_CLV_EXP_PAD 1
#endif
template <int D> struct ExpWarp { static constexpr int WARPS = D >= 8 ? 2 : 4; };   // 3 n^2 complex per warp: 12 KB at n = 16
template <typename Real, int D>
__global__ void __launch_bounds__(32 * ExpWarp<D>::WARPS) clover_exp_warp_kernel(char *clover, long vh, double m)
{
    constexpr int N2 = 2 * D, LDA = N2 + HR_CLV_EXP_PAD, NC = N2 * LDA, NE = N2 * (N2 + 1) / 2, BLK = 4 * D * D, RPV = 16 / (int)sizeof(Real), NVB = BLK / RPV;
    constexpr int WARPS = ExpWarp<D>::WARPS;
    __shared__ double2 mat[WARPS][3][NC];                          // X, E, Q
    __shared__ unsigned char rc_of[NE][2];                         // upper-triangle entry (diagonal first, then row by row) -> (r, c)
    const int warp = (int)threadIdx.x >> 5, lane = (int)threadIdx.x & 31;
    for (int e = (int)threadIdx.x; e < NE; e += (int)blockDim.x) {
        if (e < N2) { rc_of[e][0] = rc_of[e][1] = (unsigned char)e; }
        else {
            int u = e - N2, r = 0;
            while (u >= N2 - 1 - r) { u -= N2 - 1 - r; ++r; }
            rc_of[e][0] = (unsigned char)r; rc_of[e][1] = (unsigned char)(r + 1 + u);
        }
    }
    __syncthreads();
    const long blk = (long)blockIdx.x * WARPS + warp;              // over 2 parities x vh sites x 2 blocks
    if (blk >= 4 * vh) return;
    const int b = (int)(blk & 1);
    const long site = blk >> 1;
    const long par = site / vh, s = site - par * vh;
    char *rec = clover + (size_t)par * 2 * BLK * sizeof(Real) * (size_t)vh + (size_t)s * 16 + (size_t)(b * NVB) * (size_t)vh * 16;
    const size_t pb = (size_t)vh * 16;
    double2 *X = mat[warp][0], *E = mat[warp][1], *Q = mat[warp][2];
    const double sc = 1.0 / (m * 64.0);
    // packed real w of the record: w < N2 the diagonal entry w; else entry N2 + (w - N2) / 2 of rc_of, re or im
    for (int v = lane; v < NVB; v += 32) {
        Real tv[RPV];
        load_planes<LD_DEFAULT, 1>(tv, rec + (size_t)v * pb, pb, 0);
#pragma unroll
        for (int i = 0; i < RPV; ++i) {
            const int w = v * RPV + i;
            const double val = (double)tv[i] * sc;
            if (w < N2) X[w * LDA + w] = make_double2(val, 0.0);
            else {
                const int e = N2 + ((w - N2) >> 1), r = rc_of[e][0], c = rc_of[e][1];
                if (((w - N2) & 1) == 0) { X[r * LDA + c].x = val; X[c * LDA + r].x = val; }
                else { X[r * LDA + c].y = val; X[c * LDA + r].y = -val; }
            }
        }
    }
    __syncwarp();
    auto mul = [&](double2 *o, const double2 *a, const double2 *bb) {   // o = a bb, commuting Hermitian matrices
        for (int e = lane; e < NE; e += 32) {
            const int r = rc_of[e][0], c = rc_of[e][1];
            double re = 0, im = 0;
#pragma unroll
            for (int k = 0; k < N2; ++k) {
                const double2 x = a[r * LDA + k], y = bb[k * LDA + c];
                re += x.x * y.x - x.y * y.y;
                im += x.x * y.y + x.y * y.x;
            }
            if (r == c) o[r * LDA + r] = make_double2(re, 0.0);
            else { o[r * LDA + c] = make_double2(re, im); o[c * LDA + r] = make_double2(re, -im); }
        }
        __syncwarp();
    };
    for (int i = lane; i < NC; i += 32) E[i] = make_double2(X[i].x * 0.1, X[i].y * 0.1);
    __syncwarp();
    for (int k = 9; k >= 1; --k) {                                     // Horner: s_k = (X + X s_{k+1}) / k
        mul(Q, X, E);
        const double ik = 1.0 / k;
        for (int i = lane; i < NC; i += 32) E[i] = make_double2((X[i].x + Q[i].x) * ik, (X[i].y + Q[i].y) * ik);
        __syncwarp();
    }
    for (int sq = 0; sq < 6; ++sq) {                                   // expm1(2X) = expm1(X)^2 + 2 expm1(X)
        mul(Q, E, E);
        for (int i = lane; i < NC; i += 32) E[i] = make_double2(Q[i].x + 2.0 * E[i].x, Q[i].y + 2.0 * E[i].y);
        __syncwarp();
    }
    for (int v = lane; v < NVB; v += 32) {
        Real tv[RPV];
#pragma unroll
        for (int i = 0; i < RPV; ++i) {
            const int w = v * RPV + i;
            double val;
            if (w < N2) val = E[w * LDA + w].x;
            else {
                const int e = N2 + ((w - N2) >> 1), r = rc_of[e][0], c = rc_of[e][1];
                val = ((w - N2) & 1) == 0 ? E[r * LDA + c].x : E[r * LDA + c].y;
            }
            tv[i] = (Real)(m * val);
        }
        store_planes<ST_DEFAULT, 1>(rec + (size_t)v * pb, pb, tv);
    }
}

// T (or E) -> A = (4+m0) + T in place, and A^{-1} into a second field of the same layout (reading C32: the even-odd
// preconditioned operator with a clover term needs A_oo^{-1}).  One thread per (site, chirality block); the n x n
// block (n = 2 d_R <= 16) is inverted by Gauss-Jordan elimination with partial pivoting in fp64 (the inverse of a
// Hermitian matrix is Hermitian, so it packs the same way).  Set-up kernel.
// Inverse of a Hermitian POSITIVE DEFINITE n x n block in registers, every index a compile-time constant: A = L L^H
// (Cholesky, no pivoting needed for a positive definite matrix), M = L^{-1}, A^{-1} = M^H M.  Packed storage as the clover
// field: n real diagonal entries, then the strict upper triangle row by row.  Lower-triangular factors are stored at the
// transposed position: X[i][j], i > j, at up(j, i).  Returns false -- and the caller falls back to Gauss-Jordan with partial
// pivoting -- as soon as a pivot is not safely positive (A = (4+m0) + T is positive definite for any physical mass; a
// negative or tiny shifted mass makes it indefinite).
template <int N>
__device__ __forceinline__ bool hpd_inverse(const double (&ad)[N], const double (&ar)[N * (N - 1) / 2], const double (&ai)[N * (N - 1) / 2],
                                            double (&od)[N], double (&orr)[N * (N - 1) / 2], double (&oi)[N * (N - 1) / 2])
{
    constexpr int NU = N * (N - 1) / 2;
    double lr[NU], li[NU], id[N];
    bool ok = true;
#pragma unroll
    for (int j = 0; j < N; ++j) {
        double sdiag = ad[j];
#pragma unroll
        for (int k = 0; k < N; ++k)
            if (k < j) sdiag -= lr[up<N>(k, j)] * lr[up<N>(k, j)] + li[up<N>(k, j)] * li[up<N>(k, j)];
        ok = ok && (sdiag > 1e-12 * fabs(ad[j])) && (sdiag > 1e-300);
        id[j] = rsqrt(ok ? sdiag : 1.0);
#pragma unroll
        for (int i = 0; i < N; ++i)
            if (i > j) {                                           // L[i][j] = (conj(A[j][i]) - sum_k L[i][k] conj(L[j][k])) / L[j][j]
                double re = ar[up<N>(j, i)], im = -ai[up<N>(j, i)];
#pragma unroll
                for (int k = 0; k < N; ++k)
                    if (k < j) {
                        const double a = lr[up<N>(k, i)], b = li[up<N>(k, i)], c = lr[up<N>(k, j)], d = li[up<N>(k, j)];
                        re -= a * c + b * d;
                        im -= b * c - a * d;
                    }
                lr[up<N>(j, i)] = re * id[j];
                li[up<N>(j, i)] = im * id[j];
            }
    }
    if (!ok) return false;
    // M = L^{-1}: M[j][j] = 1 / L[j][j],  M[i][j] = -(1 / L[i][i]) sum_{k = j}^{i-1} L[i][k] M[k][j]
    double mr[NU], mi[NU];
#pragma unroll
    for (int j = 0; j < N; ++j)
#pragma unroll
        for (int i = 0; i < N; ++i)
            if (i > j) {
                double re = lr[up<N>(j, i)] * id[j], im = li[up<N>(j, i)] * id[j];
#pragma unroll
                for (int k = 0; k < N; ++k)
                    if (k > j && k < i) {
                        const double a = lr[up<N>(k, i)], b = li[up<N>(k, i)], c = mr[up<N>(j, k)], d = mi[up<N>(j, k)];
                        re += a * c - b * d;
                        im += a * d + b * c;
                    }
                mr[up<N>(j, i)] = -id[i] * re;
                mi[up<N>(j, i)] = -id[i] * im;
            }
    // A^{-1} = M^H M:  (r, c), r <= c:  sum_{k >= c} conj(M[k][r]) M[k][c]
#pragma unroll
    for (int r = 0; r < N; ++r) {
        double dsum = id[r] * id[r];
#pragma unroll
        for (int k = 0; k < N; ++k)
            if (k > r) dsum += mr[up<N>(r, k)] * mr[up<N>(r, k)] + mi[up<N>(r, k)] * mi[up<N>(r, k)];
        od[r] = dsum;
#pragma unroll
        for (int c = 0; c < N; ++c)
            if (c > r) {
                double re = mr[up<N>(r, c)] * id[c], im = -mi[up<N>(r, c)] * id[c];   // k = c: conj(M[c][r]) M[c][c]
#pragma unroll
                for (int k = 0; k < N; ++k)
                    if (k > c) {
                        const double a = mr[up<N>(r, k)], b = mi[up<N>(r, k)], cc = mr[up<N>(c, k)], d = mi[up<N>(c, k)];
                        re += a * cc + b * d;
                        im += a * d - b * cc;
                    }
                orr[up<N>(r, c)] = re;
                oi[up<N>(r, c)] = im;
            }
    }
    return true;
}

#ifndef HR_CLV_CHOL_MAXD
#define HR_CLV_CHOL_MAXD 4
#endif
template <typename Real, int D>
__global__ void __launch_bounds__(64) clover_finalize_kernel(char *clover, char *inverse, long vh, double m)
{
    constexpr int N2 = 2 * D, M = 2 * N2 * N2, BLK = 4 * D * D, RPV = 16 / (int)sizeof(Real), NVB = BLK / RPV;
    const long tid = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 4 * vh) return;
    const int b = (int)(tid & 1);
    const long site = tid >> 1;
    const long par = site / vh, s = site - par * vh;
    const size_t off = (size_t)par * 2 * BLK * sizeof(Real) * (size_t)vh + (size_t)s * 16 + (size_t)(b * NVB) * (size_t)vh * 16;
    const size_t pb = (size_t)vh * 16;
    Real t[BLK];
    load_planes<LD_DEFAULT, NVB>(t, clover + off, pb, 0);
    if constexpr (D <= HR_CLV_CHOL_MAXD) {
        // fast path: positive definite block, everything in registers
        constexpr int NU = N2 * (N2 - 1) / 2;
        double ad[N2], ar[NU], ai[NU], od[N2], orr[NU], oi[NU];
#pragma unroll
        for (int d = 0; d < N2; ++d) ad[d] = (double)(Real)((double)t[d] + m);      // the stored A = m + T, rounded to Real as below
#pragma unroll
        for (int e = 0; e < NU; ++e) { ar[e] = (double)t[N2 + 2 * e]; ai[e] = (double)t[N2 + 2 * e + 1]; }
        if (hpd_inverse<N2>(ad, ar, ai, od, orr, oi)) {
            Real a_out[BLK], inv_out[BLK];
#pragma unroll
            for (int d = 0; d < N2; ++d) { a_out[d] = (Real)ad[d]; inv_out[d] = (Real)od[d]; }
#pragma unroll
            for (int e = 0; e < NU; ++e) {
                a_out[N2 + 2 * e] = t[N2 + 2 * e]; a_out[N2 + 2 * e + 1] = t[N2 + 2 * e + 1];
                inv_out[N2 + 2 * e] = (Real)orr[e]; inv_out[N2 + 2 * e + 1] = (Real)oi[e];
            }
            store_planes<ST_DEFAULT, NVB>(clover + off, pb, a_out);
            store_planes<ST_DEFAULT, NVB>(inverse + off, pb, inv_out);
            return;
        }
    }
    double x[M], y[M];
    for (int i = 0; i < M; ++i) { x[i] = 0; y[i] = 0; }
    {
        int w = 0;
        for (int d = 0; d < N2; ++d) { t[w] = (Real)((double)t[w] + m); x[2 * (d * N2 + d)] = (double)t[w]; y[2 * (d * N2 + d)] = 1.0; ++w; }
        for (int r = 0; r < N2; ++r)
            for (int c = r + 1; c < N2; ++c) {
                const double re = (double)t[w++], im = (double)t[w++];
                x[2 * (r * N2 + c)] = re; x[2 * (r * N2 + c) + 1] = im;
                x[2 * (c * N2 + r)] = re; x[2 * (c * N2 + r) + 1] = -im;
            }
    }
    store_planes<ST_DEFAULT, NVB>(clover + off, pb, t);   // A = m + T
    for (int col = 0; col < N2; ++col) {
        int piv = col;
        double best = -1.0;
        for (int r = col; r < N2; ++r) {
            const double v = x[2 * (r * N2 + col)] * x[2 * (r * N2 + col)] + x[2 * (r * N2 + col) + 1] * x[2 * (r * N2 + col) + 1];
            if (v > best) { best = v; piv = r; }
        }
        if (piv != col)
            for (int k = 0; k < 2 * N2; ++k) {
                double tmp = x[2 * col * N2 + k]; x[2 * col * N2 + k] = x[2 * piv * N2 + k]; x[2 * piv * N2 + k] = tmp;
                tmp = y[2 * col * N2 + k]; y[2 * col * N2 + k] = y[2 * piv * N2 + k]; y[2 * piv * N2 + k] = tmp;
            }
        const double pr = x[2 * (col * N2 + col)], pi = x[2 * (col * N2 + col) + 1];
        const double den = pr * pr + pi * pi, ir = pr / den, ii = -pi / den; // 1 / pivot
        for (int k = 0; k < N2; ++k) {
            double re = x[2 * (col * N2 + k)], im = x[2 * (col * N2 + k) + 1];
            x[2 * (col * N2 + k)] = re * ir - im * ii; x[2 * (col * N2 + k) + 1] = re * ii + im * ir;
            re = y[2 * (col * N2 + k)]; im = y[2 * (col * N2 + k) + 1];
            y[2 * (col * N2 + k)] = re * ir - im * ii; y[2 * (col * N2 + k) + 1] = re * ii + im * ir;
        }
        for (int r = 0; r < N2; ++r) {
            if (r == col) continue;
            const double fr = x[2 * (r * N2 + col)], fi = x[2 * (r * N2 + col) + 1];
            for (int k = 0; k < N2; ++k) {
                const double ar = x[2 * (col * N2 + k)], ai = x[2 * (col * N2 + k) + 1];
                x[2 * (r * N2 + k)] -= fr * ar - fi * ai; x[2 * (r * N2 + k) + 1] -= fr * ai + fi * ar;
                const double br = y[2 * (col * N2 + k)], bi = y[2 * (col * N2 + k) + 1];
                y[2 * (r * N2 + k)] -= fr * br - fi * bi; y[2 * (r * N2 + k) + 1] -= fr * bi + fi * br;
            }
        }
    }
    {
        int w = 0;
        for (int d = 0; d < N2; ++d) t[w++] = (Real)y[2 * (d * N2 + d)];
        for (int r = 0; r < N2; ++r)
            for (int c = r + 1; c < N2; ++c) { t[w++] = (Real)y[2 * (r * N2 + c)]; t[w++] = (Real)y[2 * (r * N2 + c) + 1]; }
    }
    store_planes<ST_DEFAULT, NVB>(inverse + off, pb, t);
}

// d_R >= 6: ONE WARP per block, matrices in shared memory (the thread-per-block kernel above takes 42 ms for the sextet at
// 24^3 x 48 and 106 ms for the SU(3) adjoint).  A = (4+m0) + T is factored in place, A = L L^H (right-looking Cholesky: the
// pivot, the column scaling and the rank-1 update of the trailing triangle each shared out over the lanes), M = L^{-1} by
// forward substitution (one lane per column), A^{-1} = M^H M (upper-triangle entries over the lanes).  A block that is not
// safely positive definite is inverted by lane 0 with the pivoted Gauss-Jordan elimination of the kernel above, on the same
// shared-memory matrices (any physical mass gives positive definite blocks; the path exists for correctness).
template <int D> struct FinWarp { static constexpr int WARPS = D >= 8 ? 2 : 4; };
template <typename Real, int D>
__global__ void __launch_bounds__(32 * FinWarp<D>::WARPS) clover_finalize_warp_kernel(char *clover, char *inverse, long vh, double m)
{
    constexpr int N2 = 2 * D, LDA = N2 + 1, NC = N2 * LDA, NE = N2 * (N2 + 1) / 2, BLK = 4 * D * D, RPV = 16 / (int)sizeof(Real), NVB = BLK / RPV;
    constexpr int WARPS = FinWarp<D>::WARPS;
    __shared__ double2 mat[WARPS][2][NC];                          // A -> L (lower triangle), M / A^{-1}
    __shared__ double idiag[WARPS][N2];                            // 1 / L[j][j]
    __shared__ unsigned char rc_of[NE][2];                         // entry (diagonal first, then the upper triangle row by row) -> (r, c)
    const int warp = (int)threadIdx.x >> 5, lane = (int)threadIdx.x & 31;
    for (int e = (int)threadIdx.x; e < NE; e += (int)blockDim.x) {
        if (e < N2) { rc_of[e][0] = rc_of[e][1] = (unsigned char)e; }
        else {
            int u = e - N2, r = 0;
            while (u >= N2 - 1 - r) { u -= N2 - 1 - r; ++r; }
            rc_of[e][0] = (unsigned char)r; rc_of[e][1] = (unsigned char)(r + 1 + u);
        }
    }
    __syncthreads();
    const long blk = (long)blockIdx.x * WARPS + warp;
    if (blk >= 4 * vh) return;
    const int b = (int)(blk & 1);
    const long site = blk >> 1;
    const long par = site / vh, s = site - par * vh;
    const size_t off = (size_t)par * 2 * BLK * sizeof(Real) * (size_t)vh + (size_t)s * 16 + (size_t)(b * NVB) * (size_t)vh * 16;
    const size_t pb = (size_t)vh * 16;
    double2 *A = mat[warp][0], *Mi = mat[warp][1];
    double *id = idiag[warp];
    // load T, form A = m + T (the diagonal rounded to Real as it is stored), write A back, keep A dense in shared memory
    auto load_a = [&](bool write_back) {
        for (int v = lane; v < NVB; v += 32) {
            Real tv[RPV];
            load_planes<LD_DEFAULT, 1>(tv, clover + off + (size_t)v * pb, pb, 0);
            bool touched = false;
#pragma unroll
            for (int i = 0; i < RPV; ++i) {
                const int w = v * RPV + i;
                if (w < N2) {
                    if (write_back) { tv[i] = (Real)((double)tv[i] + m); touched = true; }
                    A[w * LDA + w] = make_double2((double)tv[i], 0.0);
                } else {
                    const int e = N2 + ((w - N2) >> 1), r = rc_of[e][0], c = rc_of[e][1];
                    const double val = (double)tv[i];
                    if (((w - N2) & 1) == 0) { A[r * LDA + c].x = val; A[c * LDA + r].x = val; }
                    else { A[r * LDA + c].y = val; A[c * LDA + r].y = -val; }
                }
            }
            if (write_back && touched) store_planes<ST_DEFAULT, 1>(clover + off + (size_t)v * pb, pb, tv);
        }
        __syncwarp();
    };
    load_a(true);
    if (lane < N2) Mi[lane * LDA + lane].x = A[lane * LDA + lane].x;   // the original diagonal, for the relative pivot test
    __syncwarp();
    bool ok = true;
    for (int j = 0; j < N2; ++j) {
        const double piv = A[j * LDA + j].x;
        ok = ok && (piv > 1e-12 * fabs(Mi[j * LDA + j].x)) && (piv > 1e-300);
        const double inv = rsqrt(ok ? piv : 1.0);
        __syncwarp();
        if (lane == 0) id[j] = inv;
        for (int i = j + 1 + lane; i < N2; i += 32) { double2 &x = A[i * LDA + j]; x.x *= inv; x.y *= inv; }   // L[i][j]
        __syncwarp();
        for (int e = lane; e < NE; e += 32) {                          // A[i][k] -= L[i][j] conj(L[k][j]),  j < k <= i
            const int k = rc_of[e][0], i = rc_of[e][1];
            if (k > j) {
                const double2 li = A[i * LDA + j], lk = A[k * LDA + j];
                double2 &x = A[i * LDA + k];
                x.x -= li.x * lk.x + li.y * lk.y;
                x.y -= li.y * lk.x - li.x * lk.y;
            }
        }
        __syncwarp();
    }
    if (ok) {
        // M = L^{-1}: lane j owns column j
        if (lane < N2) {
            const int j = lane;
            Mi[j * LDA + j] = make_double2(id[j], 0.0);
            for (int i = j + 1; i < N2; ++i) {
                double re = 0, im = 0;
                for (int k = j; k < i; ++k) {
                    const double2 l = A[i * LDA + k], x = Mi[k * LDA + j];
                    re += l.x * x.x - l.y * x.y;
                    im += l.x * x.y + l.y * x.x;
                }
                Mi[i * LDA + j] = make_double2(-id[i] * re, -id[i] * im);
            }
        }
        __syncwarp();
        // A^{-1}(r, c) = sum_{k >= c} conj(M[k][r]) M[k][c], r <= c: into the upper triangle of A's storage
        for (int e = lane; e < NE; e += 32) {
            const int r = rc_of[e][0], c = rc_of[e][1];
            double re = 0, im = 0;
            for (int k = c; k < N2; ++k) {
                const double2 x = Mi[k * LDA + r], y = Mi[k * LDA + c];
                re += x.x * y.x + x.y * y.y;
                im += x.x * y.y - x.y * y.x;
            }
            A[r * LDA + c] = make_double2(re, r == c ? 0.0 : im);       // the upper triangle of A is free (L lives below)
        }
        __syncwarp();
    } else {
        // not positive definite: Gauss-Jordan with partial pivoting by one lane (x = A, y = identity -> A^{-1}), result into A
        load_a(false);
        if (lane == 0) {
            double2 *x = A, *y = Mi;
            for (int i = 0; i < N2; ++i)
                for (int k = 0; k < N2; ++k) y[i * LDA + k] = make_double2(i == k ? 1.0 : 0.0, 0.0);
            for (int col = 0; col < N2; ++col) {
                int pv = col;
                double best = -1.0;
                for (int r = col; r < N2; ++r) {
                    const double v = x[r * LDA + col].x * x[r * LDA + col].x + x[r * LDA + col].y * x[r * LDA + col].y;
                    if (v > best) { best = v; pv = r; }
                }
                if (pv != col)
                    for (int k = 0; k < N2; ++k) {
                        double2 tmp = x[col * LDA + k]; x[col * LDA + k] = x[pv * LDA + k]; x[pv * LDA + k] = tmp;
                        tmp = y[col * LDA + k]; y[col * LDA + k] = y[pv * LDA + k]; y[pv * LDA + k] = tmp;
                    }
                const double pr = x[col * LDA + col].x, pi = x[col * LDA + col].y;
                const double den = pr * pr + pi * pi, ir = pr / den, ii = -pi / den;
                for (int k = 0; k < N2; ++k) {
                    double2 v = x[col * LDA + k];
                    x[col * LDA + k] = make_double2(v.x * ir - v.y * ii, v.x * ii + v.y * ir);
                    v = y[col * LDA + k];
                    y[col * LDA + k] = make_double2(v.x * ir - v.y * ii, v.x * ii + v.y * ir);
                }
                for (int r = 0; r < N2; ++r) {
                    if (r == col) continue;
                    const double fr = x[r * LDA + col].x, fi = x[r * LDA + col].y;
                    for (int k = 0; k < N2; ++k) {
                        const double2 av = x[col * LDA + k], bv = y[col * LDA + k];
                        x[r * LDA + k].x -= fr * av.x - fi * av.y; x[r * LDA + k].y -= fr * av.y + fi * av.x;
                        y[r * LDA + k].x -= fr * bv.x - fi * bv.y; y[r * LDA + k].y -= fr * bv.y + fi * bv.x;
                    }
                }
            }
            for (int i = 0; i < N2; ++i)
                for (int k = i; k < N2; ++k) x[i * LDA + k] = y[i * LDA + k];
        }
        __syncwarp();
    }
    for (int v = lane; v < NVB; v += 32) {
        Real tv[RPV];
#pragma unroll
        for (int i = 0; i < RPV; ++i) {
            const int w = v * RPV + i;
            double val;
            if (w < N2) val = A[w * LDA + w].x;
            else {
                const int e = N2 + ((w - N2) >> 1), r = rc_of[e][0], c = rc_of[e][1];
                val = ((w - N2) & 1) == 0 ? A[r * LDA + c].x : A[r * LDA + c].y;
            }
            tv[i] = (Real)val;
        }
        store_planes<ST_DEFAULT, 1>(inverse + off + (size_t)v * pb, pb, tv);
    }
}

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

size_t clover_nreal(const hr_ctx *c) { return (size_t)8 * c->d * c->d; }

// d_R > 4: rows of Q for a chunk of sites into a stream-ordered scratch allocation, then the packing kernel
template <typename Real, int D, bool RL, bool PLANES = false>
static hr_status build_rows(const hr_ctx *c, const CloverArgs &a, cudaStream_t st)
{
    const long total = c->V;
    // chunk sized by BYTES: 256 MiB of scratch at most (2^19 sites of d_R = 15 in fp64 were 11 GB next to the solver's
    // workspaces), so that the hand-off from the Q kernel to the packing kernel partly stays in the 126 MB L2
    const size_t per_site = (size_t)6 * 2 * D * D * sizeof(Real);
    long chunk = (long)(((size_t)256 << 20) / per_site) / 32 * 32;
    if (chunk < 32) chunk = 32;
    if (chunk > total) chunk = total;
    Real *scratch = nullptr;
    cudaError_t e = cudaMallocAsync((void **)&scratch, (size_t)chunk * 6 * 2 * D * D * sizeof(Real), st);
    if (e != cudaSuccess) { cudaGetLastError(); set_error("clover build: scratch allocation failed: %s", cudaGetErrorString(e)); return HR_ENOMEM; }
    hr_status rc = HR_OK;
    for (long first = 0; first < total && rc == HR_OK; first += chunk) {
        const long n = total - first < chunk ? total - first : chunk;
        if constexpr (PLANES) clover_plane_kernel<Real, D, RL><<<dim3((unsigned)((n + 63) / 64), 6), 64, 0, st>>>(a, scratch, first, n);
        else if constexpr (D >= 6) clover_q_staged_kernel<Real, D, RL><<<(unsigned)((n + 31) / 32), 32 * D, 0, st>>>(a, scratch, first, n);
        else clover_q_kernel<Real, D, RL><<<(unsigned)((n + 31) / 32), 32 * D, 0, st>>>(a, scratch, first, n);
        rc = launched(PLANES ? "clover_plane_kernel" : "clover_q_kernel");
        if (rc != HR_OK) break;
        if constexpr (PLANES) clover_pack_f_kernel<Real, D, RL><<<(unsigned)((n + 127) / 128), 128, 0, st>>>(a, scratch, first, n);
        else {
            constexpr int NVREC = CloverGeom<Real, D, RL>::NREAL / (16 / (int)sizeof(Real));
            clover_pack_vec_kernel<Real, D, RL><<<(unsigned)((n * NVREC + 127) / 128), 128, 0, st>>>(a, scratch, first, n);
        }
        rc = launched(PLANES ? "clover_pack_f_kernel" : "clover_pack_vec_kernel");
    }
    cudaFreeAsync(scratch, st);
    return rc;
}

hr_status launch_clover_build(const hr_ctx *c, hr_prec prec, void *clover, const void *links, double csw, cudaStream_t st)
{
    CloverArgs a;
    a.clover = clover; a.links = links; a.in = nullptr; a.out = nullptr;
    a.T = c->dims[0]; a.X = c->dims[1]; a.Y = c->dims[2]; a.Z = c->dims[3];
    a.vh = c->Vh; a.csw = csw;
    const unsigned grid = (unsigned)((c->V + 63) / 64);
    const bool rl = c->real_links != 0;
#define X(D, RL)                                                                                                      \
    if (c->d == D && rl == RL) {                                                                                      \
        if (D > 4) return prec == HR_F64 ? build_rows<double, D, RL>(c, a, st) : build_rows<float, D, RL>(c, a, st);   \
        /* plane-parallel form where it wins (measured): complex d_R = 3, and d_R = 4 */         \
        if ((D == 3 && !RL) || D == 4)                                                                                 \
            return prec == HR_F64 ? build_rows<double, (D <= 4 ? D : 2), RL, true>(c, a, st) : build_rows<float, (D <= 4 ? D : 2), RL, true>(c, a, st); \
        if (prec == HR_F64) clover_build_kernel<double, (D <= 4 ? D : 2), RL><<<grid, 64, 0, st>>>(a);               \
        else clover_build_kernel<float, (D <= 4 ? D : 2), RL><<<grid, 64, 0, st>>>(a);                               \
        return launched("clover_build_kernel");                                                                       \
    }
    X(2, false) X(3, false) X(4, false) X(6, false) X(3, true) X(8, true)
#undef X
    set_error("no clover kernel compiled for d_R=%d", c->d);
    return HR_EUNSUPPORTED;
}

#ifndef HR_CLV_EXP_WARP_MIND   // smallest d_R that takes the warp-per-block kernel
#define HR_CLV_EXP_WARP_MIND 4
#endif
hr_status launch_clover_exp(const hr_ctx *c, hr_prec prec, void *clover, double m, cudaStream_t st)
{
    const unsigned grid = (unsigned)((4 * c->Vh + 63) / 64);
#define X(D)                                                                                                          \
    if (c->d == D) {                                                                                                  \
        if (D >= HR_CLV_EXP_WARP_MIND) {                                                                              \
            constexpr int W = ExpWarp<(D >= 4 ? D : 4)>::WARPS;                                                       \
            const unsigned gw = (unsigned)((4 * c->Vh + W - 1) / W);                                                  \
            if (prec == HR_F64) clover_exp_warp_kernel<double, (D >= 4 ? D : 4)><<<gw, 32 * W, 0, st>>>((char *)clover, c->Vh, m); \
            else clover_exp_warp_kernel<float, (D >= 4 ? D : 4)><<<gw, 32 * W, 0, st>>>((char *)clover, c->Vh, m);    \
            return launched("clover_exp_warp_kernel");                                                                \
        }                                                                                                             \
        if (prec == HR_F64) clover_exp_kernel<double, (D < HR_CLV_EXP_WARP_MIND ? D : 2)><<<grid, 64, 0, st>>>((char *)clover, c->Vh, m); \
        else clover_exp_kernel<float, (D < HR_CLV_EXP_WARP_MIND ? D : 2)><<<grid, 64, 0, st>>>((char *)clover, c->Vh, m); \
        return launched("clover_exp_kernel");                                                                         \
    }
    X(2) X(3) X(4) X(6) X(8)
#undef X
    set_error("no clover kernel compiled for d_R=%d", c->d);
    return HR_EUNSUPPORTED;
}

hr_status launch_clover_finalize(const hr_ctx *c, hr_prec prec, void *clover, void *inverse, double m, cudaStream_t st)
{
    const unsigned grid = (unsigned)((4 * c->Vh + 63) / 64);
#define X(D)                                                                                                          \
    if (c->d == D) {                                                                                                  \
        if (D >= 6) {                                                                                                 \
            constexpr int W = FinWarp<(D >= 6 ? D : 6)>::WARPS;                                                       \
            const unsigned gw = (unsigned)((4 * c->Vh + W - 1) / W);                                                  \
            if (prec == HR_F64) clover_finalize_warp_kernel<double, (D >= 6 ? D : 6)><<<gw, 32 * W, 0, st>>>((char *)clover, (char *)inverse, c->Vh, m); \
            else clover_finalize_warp_kernel<float, (D >= 6 ? D : 6)><<<gw, 32 * W, 0, st>>>((char *)clover, (char *)inverse, c->Vh, m); \
            return launched("clover_finalize_warp_kernel");                                                           \
        }                                                                                                             \
        if (prec == HR_F64) clover_finalize_kernel<double, (D < 6 ? D : 2)><<<grid, 64, 0, st>>>((char *)clover, (char *)inverse, c->Vh, m); \
        else clover_finalize_kernel<float, (D < 6 ? D : 2)><<<grid, 64, 0, st>>>((char *)clover, (char *)inverse, c->Vh, m); \
        return launched("clover_finalize_kernel");                                                                    \
    }
    X(2) X(3) X(4) X(6) X(8)
#undef X
    set_error("no clover kernel compiled for d_R=%d", c->d);
    return HR_EUNSUPPORTED;
}

// out (+)= T in on one parity; mode +1: out += T in, 0: out = T in, -1: out = T in - out
hr_status launch_clover_apply(const hr_ctx *c, hr_prec prec, void *out, const void *in, const void *clover_parity, cudaStream_t st, int mode)
{
    CloverArgs a;
    a.clover = const_cast<void *>(clover_parity); a.links = nullptr; a.in = in; a.out = out;
    a.T = c->dims[0]; a.X = c->dims[1]; a.Y = c->dims[2]; a.Z = c->dims[3];
    a.vh = c->Vh; a.csw = 0;
    const unsigned grid = (unsigned)((2 * c->Vh + 127) / 128);
#define GO(Real, D)                                                                                                   \
    do {                                                                                                              \
        if (mode > 0) clover_apply_kernel<Real, D, 1><<<grid, 128, 0, st>>>(a);                                      \
        else if (mode == 0) clover_apply_kernel<Real, D, 0><<<grid, 128, 0, st>>>(a);                                \
        else clover_apply_kernel<Real, D, -1><<<grid, 128, 0, st>>>(a);                                              \
    } while (0)
#define X(D)                                                                                                          \
    if (c->d == D) {                                                                                                  \
        if (prec == HR_F64) GO(double, D); else GO(float, D);                                                         \
        return launched("clover_apply_kernel");                                                                       \
    }
    X(2) X(3) X(4) X(6) X(8)
#undef X
#undef GO
    set_error("no clover kernel compiled for d_R=%d", c->d);
    return HR_EUNSUPPORTED;
}

} // namespace hr
