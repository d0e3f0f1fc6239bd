// dphi_kernel.cuh -- the even-odd Wilson hopping term for sm_100a.
//
//   out(x) = -1/2 sum_mu [ (1-gamma_mu) s+ U_mu(x) psi(x+mu) + (1+gamma_mu) s- U_mu(x-mu)^dag psi(x-mu) ]
//            (+ (4+m0) psi(x) when MASS)                                  BASELINE.json:north_star
//
// Design:
//  * a3  site -> coordinates -> 8 neighbour half-indices and seam signs by integer arithmetic in the
//        kernel; no neighbour tables, no halo (north_star: "periodic/antiperiodic boundaries resolved by
//        in-kernel index arithmetic").
//  * a4  spin projection to a half spinor BEFORE the colour multiply (the paper's half-spinor idea,
//        PAPER.md:64, moved inside the kernel).  In the chiral basis of reading C1 every projector has
//        the form   h_k = psi_k + c_k psi_{p(k)},  k = 0,1,  c_k in {+-1, +-i},
//        and the reconstruction is   out_k += chi_k,  out_{p(k)} += conj(c_k) chi_k :
//            mu   p(0) p(1)   c_0 (forward)  c_1 (forward)       (backward: both negated)
//            0     2    3        1              1
//            1     3    2        i              i
//            2     3    2        1             -1
//            3     2    3        i             -i
//        so the whole spin algebra is additions; the seam sign rides on the FMA that accumulates chi.
//  * a5  colour multiply chi_k = U h_k / U^dagger h_k with the d_R x d_R link (real for the adjoint),
//        fully unrolled on compile-time D.
//  * a6  accumulate, scale by -1/2, optional (4+m0) psi(x), store.
//  * KSPLIT = 1: one thread per site.  KSPLIT = 2: two threads per site, thread k owns half-spinor
//        component k (loads psi_k and psi_{p(k)}: no redundant spinor traffic; both lanes read the same
//        link addresses, which the coalescer merges) -- the register-pressure answer to the paper's
//        large-N_f problem at d_R >= 6.
//  * loads are 128-bit, coalesced over the half index (hr_internal.h); links are streamed past L1
//        (and optionally evict-first in L2), neighbour spinors are left to L1/L2 for re-use.
#pragma once
#include <type_traits>

#include "hr_internal.h"

// HR_PDL: the one-thread-per-site / pair kernels are launched with programmatic stream serialization, so that back-to-back
// Dphi launches overlap the launch latency of one with the tail of the other (small lattices: "dominated by the
// kernel call overheads")
#ifndef HR_PDL
#define HR_PDL 1
#endif
#include "packed_f32.cuh"

namespace hr {

template <int CRE, int CIM, typename Real>
__device__ __forceinline__ void add_c(Real &ore, Real &oim, Real are, Real aim, Real bre, Real bim, Real sk)
{
    // o = a + sk * c * b,  c = CRE + i CIM, exactly one of CRE, CIM non-zero, sk = +-1 (real)
    if constexpr (CRE != 0) {
        ore = fma((Real)CRE * sk, bre, are);
        oim = fma((Real)CRE * sk, bim, aim);
    } else {
        ore = fma((Real)(-CIM) * sk, bim, are);
        oim = fma((Real)CIM * sk, bre, aim);
    }
}

template <int CRE, int CIM, typename Real>
__device__ __forceinline__ void acc_conj_c(Real &ore, Real &oim, Real xre, Real xim, Real w)
{
    // o += w * conj(c) * x,  conj(c) = CRE - i CIM
    if constexpr (CRE != 0) {
        ore = fma((Real)CRE * w, xre, ore);
        oim = fma((Real)CRE * w, xim, oim);
    } else {
        ore = fma((Real)CIM * w, xim, ore);
        oim = fma((Real)(-CIM) * w, xre, oim);
    }
}

// chi = U h (DAG = false) or U^dagger h (DAG = true); U complex [D][D] (re,im) or real [D][LDM] (LDM: row stride, LinkGeom::LD)
template <int D, bool RL, bool DAG, typename Real, int LDM = D>
__device__ __forceinline__ void colour_mul(Real (&chi)[2 * D], const Real *u, const Real (&h)[2 * D])
{
    static_assert(RL || LDM == D, "padded rows: real links only");
#pragma unroll
    for (int i = 0; i < D; ++i) {
        Real re = 0, im = 0;
#pragma unroll
        for (int j = 0; j < D; ++j) {
            if constexpr (RL) {
                const Real r = DAG ? u[j * LDM + i] : u[i * LDM + j];
                re = fma(r, h[2 * j], re);
                im = fma(r, h[2 * j + 1], im);
            } else {
                const int e = DAG ? 2 * (j * D + i) : 2 * (i * D + j);
                const Real ur = u[e], ui = u[e + 1];
                if constexpr (!DAG) {
                    re = fma(ur, h[2 * j], re);
                    re = fma(-ui, h[2 * j + 1], re);
                    im = fma(ur, h[2 * j + 1], im);
                    im = fma(ui, h[2 * j], im);
                } else {
                    re = fma(ur, h[2 * j], re);
                    re = fma(ui, h[2 * j + 1], re);
                    im = fma(ur, h[2 * j + 1], im);
                    im = fma(-ui, h[2 * j], im);
                }
            }
        }
        chi[2 * i] = re;
        chi[2 * i + 1] = im;
    }
}

// ---- link kinds ------------------------------------------------------------------------------------
// LK_COMPLEX / LK_REAL: the represented d_R x d_R link is read from memory (hr_represent_links wrote it).
// LK_SYM_OTF / LK_ASYM_OTF ("on-the-fly representation"): the kernel reads the
// FUNDAMENTAL N x N link (144 B instead of 576 B for the SU(3) sextet in fp64) and applies the two-index
// representation without ever forming R(U): with the colour vector written as the (anti)symmetric matrix
// Psi = sum_a psi_a e_a (basis of reading C8),  R(U) psi <-> U Psi U^T  and  R(U)^dagger psi <-> U^dagger Psi U^*.
// LK_ROWS / LK_ADJ2_ROWS: the fundamental link is stored as its first N-1 rows (SU(3): 12 of 18 reals, SU(2): 4 of 8);
// the last row is rebuilt in registers (SU(3): conj(row0 x row1); SU(2): (-conj u01, conj u00)) -- 25-33 % fewer
// link bytes for the fundamental representation.  LK_ADJ2_ROWS builds the real 3x3 SU(2) adjoint link from the four
// reals (a0, a3, a2, a1) = first row of U = a0 + i a.sigma:  R_ab = (a0^2 - a.a) delta_ab + 2 a_a a_b + 2 a0 eps_abc a_c
// (32 B instead of 72 B per link in fp64).  Valid for links that ARE special unitary (reading C30).
// LK_ADJ3_OTF / LK_ADJ3_ROWS: the SU(3) ADJOINT (d_R = 8) applied on the fly from the fundamental link (18 reals, or its
// first two rows): with Psi = sum_a psi_a T_a (T_a = lambda_a/2, nested Gell-Mann order of reading C6),
// (R psi)_a = 2 tr(T_a U Psi U^dagger) and (R^T psi)_a = 2 tr(T_a U^dagger Psi U) -- the 8 x 8 real link (512 B in
// fp64, the paper's large-N_f register problem) is never formed: 144 or 96 B are read instead.
enum : int { LK_COMPLEX = 0, LK_REAL = 1, LK_SYM_OTF = 2, LK_ASYM_OTF = 3, LK_ROWS = 4, LK_ADJ2_ROWS = 5, LK_ADJ3_OTF = 6,
             LK_ADJ3_ROWS = 7 };

template <int LK, int D> struct LinkGeom {
    // N of the fundamental link for the on-the-fly kinds: D = N(N+1)/2 (sym) or N(N-1)/2 (asym)
    static constexpr int N = LK == LK_SYM_OTF ? (D == 3 ? 2 : D == 6 ? 3 : D == 10 ? 4 : 0)
                           : LK == LK_ASYM_OTF ? (D == 3 ? 3 : D == 6 ? 4 : 0)
                           : LK == LK_ADJ2_ROWS ? (D == 3 ? 2 : 0)
                           : (LK == LK_ADJ3_OTF || LK == LK_ADJ3_ROWS) ? (D == 8 ? 3 : 0) : D;
    // row stride of the represented real link: d_R + 1 for an odd d_R > 8 (hr_internal.h link_ld), the extra entry is zero
    static constexpr int LD = (LK == LK_REAL && (D & 1) && D > 8) ? D + 1 : D;
    static constexpr int NREAL = LK == LK_REAL ? D * LD : LK == LK_COMPLEX ? 2 * D * D
                               : (LK == LK_ROWS || LK == LK_ADJ2_ROWS || LK == LK_ADJ3_ROWS) ? 2 * N * (N - 1) : 2 * N * N;
    static_assert(N > 0, "no such two-index representation");
};

// chi = R(U) h (DAG = false) or R(U)^dagger h (DAG = true) from the fundamental link u[N][N] (re,im)
template <int D, int LK, bool DAG, typename Real>
__device__ __forceinline__ void twoindex_mul(Real (&chi)[2 * D], const Real *u, const Real (&h)[2 * D])
{
    constexpr int N = LinkGeom<LK, D>::N;
    constexpr bool SYM = LK == LK_SYM_OTF;
    // Psi' = sqrt2 * Psi: off-diagonal entries are the components themselves, diagonal ones (sym only) sqrt2 * h;
    // then chi_(ij) = M'_ij (i<j), chi_(ii) = M'_ii / sqrt2 with M' = U Psi' U^T.
    Real pr[N][N], pi[N][N];
    {
        int a = 0;
#pragma unroll
        for (int i = 0; i < N; ++i)
#pragma unroll
            for (int j = i; j < N; ++j) {
                if (i == j) {
                    if constexpr (SYM) { pr[i][i] = (Real)1.4142135623730951 * h[2 * a]; pi[i][i] = (Real)1.4142135623730951 * h[2 * a + 1]; ++a; }
                    else { pr[i][i] = 0; pi[i][i] = 0; }
                } else {
                    pr[i][j] = h[2 * a]; pi[i][j] = h[2 * a + 1];
                    pr[j][i] = SYM ? h[2 * a] : -h[2 * a]; pi[j][i] = SYM ? h[2 * a + 1] : -h[2 * a + 1];
                    ++a;
                }
            }
    }
    // W = U (or U^dagger):  wr/wi[i][k], the imaginary part conjugated for the dagger
    auto wr = [&](int i, int k) -> Real { return DAG ? u[2 * (k * N + i)] : u[2 * (i * N + k)]; };
    auto wi = [&](int i, int k) -> Real { return DAG ? -u[2 * (k * N + i) + 1] : u[2 * (i * N + k) + 1]; };
    // row by row:  A_i. = (W Psi')_i.  is used at once for  M'_ij = sum_l A_il W_jl  (j >= i: M' is (anti)symmetric), so only
    // one row of A is ever live -- 2N reals instead of 2N^2 (the register budget of this kernel is what limits its warps)
    int a = 0;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        Real ar[N], ai[N];
#pragma unroll
        for (int l = 0; l < N; ++l) {
            Real re = 0, im = 0;
#pragma unroll
            for (int k = 0; k < N; ++k) {
                if (!SYM && k == l) continue;
                re = fma(wr(i, k), pr[k][l], re); re = fma(-wi(i, k), pi[k][l], re);
                im = fma(wr(i, k), pi[k][l], im); im = fma(wi(i, k), pr[k][l], im);
            }
            ar[l] = re; ai[l] = im;
        }
#pragma unroll
        for (int j = i; j < N; ++j) {
            if (!SYM && i == j) continue;
            Real re = 0, im = 0;
#pragma unroll
            for (int l = 0; l < N; ++l) {
                re = fma(ar[l], wr(j, l), re); re = fma(-ai[l], wi(j, l), re);
                im = fma(ar[l], wi(j, l), im); im = fma(ai[l], wr(j, l), im);
            }
            if (i == j) { re *= (Real)0.7071067811865476; im *= (Real)0.7071067811865476; }
            chi[2 * a] = re; chi[2 * a + 1] = im;
            ++a;
        }
    }
}

// full N x N complex link from its first N-1 rows (N = 2, 3)
template <int N, typename Real> __device__ __forceinline__ void rebuild_rows(Real (&f)[2 * N * N], const Real *r)
{
    static_assert(N == 2 || N == 3, "row reconstruction for SU(2) and SU(3)");
#pragma unroll
    for (int e = 0; e < 2 * N * (N - 1); ++e) f[e] = r[e];
    if constexpr (N == 2) {
        f[4] = -r[2]; f[5] = r[3];   // -conj(u01)
        f[6] = r[0];  f[7] = -r[1];  //  conj(u00)
    } else {
        // row2_j = conj(row0_k row1_l - row0_l row1_k), (j,k,l) cyclic
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const int k = (j + 1) % 3, l = (j + 2) % 3;
            const Real ar = r[2 * k], ai = r[2 * k + 1], br = r[6 + 2 * l], bi = r[6 + 2 * l + 1];
            const Real cr = r[2 * l], ci = r[2 * l + 1], dr = r[6 + 2 * k], di = r[6 + 2 * k + 1];
            f[12 + 2 * j] = (ar * br - ai * bi) - (cr * dr - ci * di);
            f[12 + 2 * j + 1] = -((ar * bi + ai * br) - (cr * di + ci * dr));
        }
    }
}

// real 3x3 SU(2) adjoint link from (a0, a3, a2, a1) = the first row of the fundamental link
template <typename Real> __device__ __forceinline__ void rebuild_adj2(Real (&m)[9], const Real *r)
{
    const Real a0 = r[0], a[3] = { r[3], r[2], r[1] };
    const Real dg = a0 * a0 - (a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) m[3 * i + j] = (Real)2 * a[i] * a[j] + (i == j ? dg : (Real)0);
    // + 2 a0 eps_ijk a_k
    m[1] += (Real)2 * a0 * a[2]; m[3] -= (Real)2 * a0 * a[2];
    m[5] += (Real)2 * a0 * a[0]; m[7] -= (Real)2 * a0 * a[0];
    m[6] += (Real)2 * a0 * a[1]; m[2] -= (Real)2 * a0 * a[1];
}

// chi = R^adj(U) h (DAG = false) or R^adj(U)^T h (DAG = true) for SU(3), from the fundamental link u[3][3] (re,im);
// components in the nested Gell-Mann order: 0 S01, 1 A01, 2 D1, 3 S02, 4 A02, 5 S12, 6 A12, 7 D2
template <bool DAG, typename Real>
__device__ __forceinline__ void adj3_mul(Real (&chi)[16], const Real *u, const Real (&h)[16])
{
    constexpr Real IS3 = (Real)0.57735026918962576451; // 1/sqrt(3)
    // Psi = (1/2) sum_a h_a lambda_a  (the factor 1/2 is applied at the end together with the 2 of 2 tr(T_a .))
    Real pr[3][3], pi[3][3];
    auto offd = [&](int i, int m, int s, int a) { // Psi_im = h_S - i h_A, Psi_mi = h_S + i h_A
        pr[i][m] = h[2 * s] + h[2 * a + 1]; pi[i][m] = h[2 * s + 1] - h[2 * a];
        pr[m][i] = h[2 * s] - h[2 * a + 1]; pi[m][i] = h[2 * s + 1] + h[2 * a];
    };
    offd(0, 1, 0, 1); offd(0, 2, 3, 4); offd(1, 2, 5, 6);
    pr[0][0] = h[4] + IS3 * h[14]; pi[0][0] = h[5] + IS3 * h[15];
    pr[1][1] = -h[4] + IS3 * h[14]; pi[1][1] = -h[5] + IS3 * h[15];
    pr[2][2] = (Real)-2 * IS3 * h[14]; pi[2][2] = (Real)-2 * IS3 * h[15];
    auto wr = [&](int i, int k) -> Real { return DAG ? u[2 * (k * 3 + i)] : u[2 * (i * 3 + k)]; };
    auto wi = [&](int i, int k) -> Real { return DAG ? -u[2 * (k * 3 + i) + 1] : u[2 * (i * 3 + k) + 1]; };
    Real ar[3][3], ai[3][3], mr[3][3], mi[3][3];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int l = 0; l < 3; ++l) {
            Real re = 0, im = 0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                re = fma(wr(i, k), pr[k][l], re); re = fma(-wi(i, k), pi[k][l], re);
                im = fma(wr(i, k), pi[k][l], im); im = fma(wi(i, k), pr[k][l], im);
            }
            ar[i][l] = re; ai[i][l] = im;
        }
    // M = A W^dagger: M_ij = sum_l A_il conj(W_jl)
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            Real re = 0, im = 0;
#pragma unroll
            for (int l = 0; l < 3; ++l) {
                re = fma(ar[i][l], wr(j, l), re); re = fma(ai[i][l], wi(j, l), re);
                im = fma(ai[i][l], wr(j, l), im); im = fma(-ar[i][l], wi(j, l), im);
            }
            mr[i][j] = re; mi[i][j] = im;
        }
    // chi_a = tr(lambda_a M) / 2 ... with Psi carrying no 1/2: chi_a = (1/2) tr(lambda_a M)
    auto ext = [&](int i, int m, int s, int a) {
        chi[2 * s] = (Real)0.5 * (mr[m][i] + mr[i][m]); chi[2 * s + 1] = (Real)0.5 * (mi[m][i] + mi[i][m]);
        // i (M_im - M_mi)
        chi[2 * a] = (Real)-0.5 * (mi[i][m] - mi[m][i]); chi[2 * a + 1] = (Real)0.5 * (mr[i][m] - mr[m][i]);
    };
    ext(0, 1, 0, 1); ext(0, 2, 3, 4); ext(1, 2, 5, 6);
    chi[4] = (Real)0.5 * (mr[0][0] - mr[1][1]); chi[5] = (Real)0.5 * (mi[0][0] - mi[1][1]);
    chi[14] = (Real)0.5 * IS3 * (mr[0][0] + mr[1][1] - (Real)2 * mr[2][2]);
    chi[15] = (Real)0.5 * IS3 * (mi[0][0] + mi[1][1] - (Real)2 * mi[2][2]);
}

template <int D, int LK, bool DAG, typename Real>
__device__ __forceinline__ void link_mul(Real (&chi)[2 * D], const Real *u, const Real (&h)[2 * D])
{
    if constexpr (LK == LK_COMPLEX || LK == LK_REAL) colour_mul<D, LK == LK_REAL, DAG, Real, LinkGeom<LK, D>::LD>(chi, u, h);
    else if constexpr (LK == LK_ROWS) {
        Real f[2 * D * D];
        rebuild_rows<D>(f, u);     // identical for both half-spinor components of a hop: the compiler merges the two
        colour_mul<D, false, DAG>(chi, f, h);
    } else if constexpr (LK == LK_ADJ2_ROWS) {
        Real m[9];
        rebuild_adj2(m, u);
        colour_mul<3, true, DAG>(chi, m, h);
    } else if constexpr (LK == LK_ADJ3_OTF) {
        adj3_mul<DAG>(chi, u, h);
    } else if constexpr (LK == LK_ADJ3_ROWS) {
        Real f[18];
        rebuild_rows<3>(f, u);
        adj3_mul<DAG>(chi, f, h);
    } else twoindex_mul<D, LK, DAG>(chi, u, h);
}

// Run `f(kind, link)` with the link in the form the colour multiply wants: row-compressed kinds are rebuilt ONCE per
// hop here (both half-spinor components then share the registers), every other kind is passed through.
template <int D, int LK, typename Real, typename F>
__device__ __forceinline__ void with_link(const Real *u, F &&f)
{
    if constexpr (LK == LK_ROWS) {
        Real full[2 * D * D];
        rebuild_rows<D>(full, u);
        f(std::integral_constant<int, LK_COMPLEX>{}, (const Real *)full);
    } else if constexpr (LK == LK_ADJ2_ROWS) {
        Real m[9];
        rebuild_adj2(m, u);
        f(std::integral_constant<int, LK_REAL>{}, (const Real *)m);
    } else if constexpr (LK == LK_ADJ3_ROWS) {
        Real full[18];
        rebuild_rows<3>(full, u);
        f(std::integral_constant<int, LK_ADJ3_OTF>{}, (const Real *)full);
    } else {
        f(std::integral_constant<int, LK>{}, u);
    }
}

// one half-spinor component of one hop:  h = a + sk c0 b ; chi = U(^dag) h ; outK += sgn chi ;
// outP += sgn sk conj(c0) chi.   c0 = (DIR ? -1 : +1) * (MU in {0,2} ? 1 : i)
template <int MU, int DIR, int D, int LK, typename Real>
__device__ __forceinline__ void hop_component(const Real *u, const Real *a, const Real *b, Real sk, Real sgn,
                                              Real *outK, Real *outP)
{
    constexpr int S = DIR ? -1 : 1;
    constexpr int CRE = (MU == 0 || MU == 2) ? S : 0;
    constexpr int CIM = (MU == 0 || MU == 2) ? 0 : S;
    Real h[2 * D], chi[2 * D];
#pragma unroll
    for (int c = 0; c < D; ++c) add_c<CRE, CIM>(h[2 * c], h[2 * c + 1], a[2 * c], a[2 * c + 1], b[2 * c], b[2 * c + 1], sk);
    link_mul<D, LK, DIR == 1>(chi, u, h);
    const Real w = sgn * sk;
#pragma unroll
    for (int c = 0; c < D; ++c) {
        outK[2 * c] = fma(sgn, chi[2 * c], outK[2 * c]);
        outK[2 * c + 1] = fma(sgn, chi[2 * c + 1], outK[2 * c + 1]);
        acc_conj_c<CRE, CIM>(outP[2 * c], outP[2 * c + 1], chi[2 * c], chi[2 * c + 1], w);
    }
}

// Both half-spinor components of one hop at once, for fp32: component 0 in lane 0 and component 1 in lane 1 of packed
// registers, the link broadcast to both lanes -- the link multiply then runs on FFMA2 / FADD2 / FMUL2 (packed_f32.cuh) at
// half the instruction count.  The projections before and the accumulations after stay scalar: a scalar result can be
// written straight into either half of a register pair, so packing and unpacking cost no instruction.
#ifndef HR_PACK32
#define HR_PACK32 1
#endif
template <int LK, typename Real> struct PackedHop {
    // the kinds whose link multiply is arithmetic-bound in fp32: the representations applied on the fly
    static constexpr bool value = HR_PACK32 && sizeof(Real) == 4 &&
                                  (LK == LK_SYM_OTF || LK == LK_ASYM_OTF || LK == LK_ADJ3_OTF || LK == LK_ADJ3_ROWS);
};

template <int MU, int DIR, int D, int LK>
__device__ __forceinline__ void hop_pair_packed(const float *u, const float *psi, float sgn, float (&acc)[4][2 * D])
{
    using pk::f32x2;
    constexpr int S = DIR ? -1 : 1;
    constexpr int CRE = (MU == 0 || MU == 2) ? S : 0;
    constexpr int CIM = (MU == 0 || MU == 2) ? 0 : S;
    constexpr int P0 = (MU == 0 || MU == 3) ? 2 : 3;
    constexpr int P1 = 5 - P0;
    constexpr float SK1 = MU >= 2 ? -1.f : 1.f;
    constexpr int NL = LinkGeom<LK, D>::NREAL;
    f32x2 up[NL], hp[2 * D], chip[2 * D];
#pragma unroll
    for (int e = 0; e < NL; ++e) up[e] = f32x2(u[e]);
#pragma unroll
    for (int c = 0; c < D; ++c) {
        float h0r, h0i, h1r, h1i;
        add_c<CRE, CIM>(h0r, h0i, psi[2 * c], psi[2 * c + 1], psi[P0 * 2 * D + 2 * c], psi[P0 * 2 * D + 2 * c + 1], 1.f);
        add_c<CRE, CIM>(h1r, h1i, psi[2 * D + 2 * c], psi[2 * D + 2 * c + 1], psi[P1 * 2 * D + 2 * c], psi[P1 * 2 * D + 2 * c + 1], SK1);
        hp[2 * c] = f32x2(h0r, h1r);
        hp[2 * c + 1] = f32x2(h0i, h1i);
    }
    link_mul<D, LK, DIR == 1, f32x2>(chip, up, hp);
    const float w1 = sgn * SK1;
#pragma unroll
    for (int c = 0; c < D; ++c) {
        const float c0r = chip[2 * c].v.x, c0i = chip[2 * c + 1].v.x, c1r = chip[2 * c].v.y, c1i = chip[2 * c + 1].v.y;
        acc[0][2 * c] = fma(sgn, c0r, acc[0][2 * c]);
        acc[0][2 * c + 1] = fma(sgn, c0i, acc[0][2 * c + 1]);
        acc[1][2 * c] = fma(sgn, c1r, acc[1][2 * c]);
        acc[1][2 * c + 1] = fma(sgn, c1i, acc[1][2 * c + 1]);
        acc_conj_c<CRE, CIM>(acc[P0][2 * c], acc[P0][2 * c + 1], c0r, c0i, sgn);
        acc_conj_c<CRE, CIM>(acc[P1][2 * c], acc[P1][2 * c + 1], c1r, c1i, w1);
    }
}

// epilogue coefficients in the kernel's precision, straight from the constant bank
template <typename Real> __device__ __forceinline__ Real coef_alpha(const DphiArgs &a, int i);
template <> __device__ __forceinline__ double coef_alpha<double>(const DphiArgs &a, int i) { return a.alpha[i]; }
template <> __device__ __forceinline__ float coef_alpha<float>(const DphiArgs &a, int i) { return a.alphaf[i]; }
template <typename Real> __device__ __forceinline__ Real coef_beta(const DphiArgs &a, int i);
template <> __device__ __forceinline__ double coef_beta<double>(const DphiArgs &a, int i) { return a.beta[i]; }
template <> __device__ __forceinline__ float coef_beta<float>(const DphiArgs &a, int i) { return a.betaf[i]; }

// w += M v for the site-diagonal matrix M of one site (two packed Hermitian 2D x 2D blocks, clover.cu layout), streamed
// one 16-byte vector at a time; v, w: the site's spinor [spin][colour] (re, im)
template <typename Real, int D>
__device__ __forceinline__ void site_matvec(Real (&w)[8 * D], const Real (&v)[8 * D], const char *mat, size_t vh, size_t s)
{
    constexpr int BLK = 4 * D * D, N2 = 2 * D, RPV = 16 / (int)sizeof(Real), NVB = BLK / RPV;
    const size_t pb = vh * 16;
#pragma unroll
    for (int b = 0; b < 2; ++b) {
        const char *tp = mat + s * 16 + (size_t)(b * NVB) * pb;
        const int o = b * 2 * N2;
        Real tv[RPV];
        int idx = 0;
        auto next = [&]() -> Real {
            if (idx % RPV == 0) load_planes<LD_STREAM, 1>(tv, tp + (size_t)(idx / RPV) * pb, pb, 0);
            return tv[idx++ % RPV];
        };
#pragma unroll
        for (int d = 0; d < N2; ++d) {
            const Real t = next();
            w[o + 2 * d] = fma(t, v[o + 2 * d], w[o + 2 * d]);
            w[o + 2 * d + 1] = fma(t, v[o + 2 * d + 1], w[o + 2 * d + 1]);
        }
#pragma unroll
        for (int r = 0; r < N2; ++r)
#pragma unroll
            for (int c = r + 1; c < N2; ++c) {
                const Real re = next();
                const Real im = next();
                w[o + 2 * r] = fma(re, v[o + 2 * c], fma(-im, v[o + 2 * c + 1], w[o + 2 * r]));
                w[o + 2 * r + 1] = fma(re, v[o + 2 * c + 1], fma(im, v[o + 2 * c], w[o + 2 * r + 1]));
                w[o + 2 * c] = fma(re, v[o + 2 * r], fma(im, v[o + 2 * r + 1], w[o + 2 * c]));
                w[o + 2 * c + 1] = fma(re, v[o + 2 * r + 1], fma(-im, v[o + 2 * r], w[o + 2 * c + 1]));
            }
    }
}

struct SiteGeom {
    int t, x, y, zh, b; // b = offset bit: z = 2*zh + b
};

// neighbour half index and seam sign of the hop (MU, DIR) from the site with half index s
template <int MU, int DIR>
__device__ __forceinline__ void neighbour(const DphiArgs &a, const SiteGeom &g, long s, long &sn, int &sign)
{
    const long sy = a.Zh, sx = (long)a.Y * a.Zh, st = (long)a.X * a.Y * a.Zh;
    if constexpr (MU == 0) {
        if constexpr (DIR == 0) { const bool w = g.t == a.T - 1; sn = w ? s - (a.T - 1) * st : s + st; sign = w ? a.bc[0] : 1; }
        else                    { const bool w = g.t == 0;       sn = w ? s + (a.T - 1) * st : s - st; sign = w ? a.bc[0] : 1; }
    } else if constexpr (MU == 1) {
        if constexpr (DIR == 0) { const bool w = g.x == a.X - 1; sn = w ? s - (a.X - 1) * sx : s + sx; sign = w ? a.bc[1] : 1; }
        else                    { const bool w = g.x == 0;       sn = w ? s + (a.X - 1) * sx : s - sx; sign = w ? a.bc[1] : 1; }
    } else if constexpr (MU == 2) {
        if constexpr (DIR == 0) { const bool w = g.y == a.Y - 1; sn = w ? s - (a.Y - 1) * sy : s + sy; sign = w ? a.bc[2] : 1; }
        else                    { const bool w = g.y == 0;       sn = w ? s + (a.Y - 1) * sy : s - sy; sign = w ? a.bc[2] : 1; }
    } else {
        // z = 2 zh + b; the neighbour row has offset bit 1-b
        if constexpr (DIR == 0) {
            const bool w = g.zh == a.Zh - 1;
            sn = g.b ? (w ? s - (a.Zh - 1) : s + 1) : s;
            sign = (g.b && w) ? a.bc[3] : 1;
        } else {
            const bool w = g.zh == 0;
            sn = g.b ? s : (w ? s + (a.Zh - 1) : s - 1);
            sign = (!g.b && w) ? a.bc[3] : 1;
        }
    }
}

// MASS: the epilogue reads self = psi(x) on the output parity (alpha term); RED: the epilogue also
// reduces sum |out|^2 and <self, out> over the launch (needs MASS) -- what a CG on gamma5 Dhat needs
// from its operator, with no extra pass over the fields.
// CLV: a site-diagonal matrix fused into the epilogue (DphiArgs::site_mode): 1 adds M self (needs MASS), 2 applies M to
// the scaled hop sum; one-thread-per-site kernels only.
template <typename Real, int D, int LK, int KSPLIT, bool MASS, bool RED, int LHINT, int SHINT, int STHINT, int MAXT, int MINB, int CLV = 0>
__global__ void __launch_bounds__(MAXT, MINB) dphi_kernel(const DphiArgs a)
{
    static_assert(!RED || MASS, "the fused reduction needs the self field");
    static_assert(CLV == 0 || (KSPLIT == 1 && !RED && (CLV != 1 || MASS) && (CLV != 2 || !MASS)), "fused site matrix: site kernels only");
#if HR_PDL
    // programmatic dependent launch (launch_one sets the stream-serialization attribute): this grid may be SCHEDULED while
    // the previous kernel of the stream is still draining; nothing is read or written before the wait, which returns when
    // that kernel has completed and its memory operations are visible.  launch_dependents lets the NEXT kernel do the same.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;");
#endif
    if (a.skip != nullptr && *a.skip != 0) return;
    constexpr int LNREAL = LinkGeom<LK, D>::NREAL;         // reals per link record read by the kernel
    constexpr int RPV = 16 / (int)sizeof(Real);
    constexpr int SPV = 2 * D / RPV;                       // 16-byte vectors per spin component
    static_assert(KSPLIT == 1 || (2 * D) % RPV == 0, "KSPLIT=2 needs vector-aligned spin components");
    constexpr size_t LB = (size_t)LNREAL * sizeof(Real);  // link bytes per site

    const long tid = (long)blockIdx.x * blockDim.x + threadIdx.x;
    long s = tid / KSPLIT;
    const int k = (int)(tid % KSPLIT);
    const bool live = s < a.nsite;
    if (!live) s = a.nsite - 1; // keep the pair convergent for the final shuffle; stores are predicated

    // Thread order -> site (a3).  Threads walk the lattice as [x / Xb][t][x % Xb][y][zh] while the
    // storage order stays [t][x][y][zh]: the +-t neighbours of a site are then Xb*Y*Zh threads away
    // instead of X*Y*Zh, so the spinors (and nothing else) that one t-slice of an x-block loads are
    // still in L2 when the next t-slice needs them.  Xb = X is the identity order.
    SiteGeom g;
    {
        unsigned r = (unsigned)s; // Vh < 2^31 (hr_ctx_create)
        g.zh = (int)(r % (unsigned)a.Zh); r /= (unsigned)a.Zh;
        g.y = (int)(r % (unsigned)a.Y); r /= (unsigned)a.Y;
        const int xl = (int)(r % (unsigned)a.Xb); r /= (unsigned)a.Xb;
        g.t = a.t0 + (int)(r % (unsigned)a.Tl);              // the launch covers the slices [t0, t0 + Tl): all of them, or a chunk
        g.x = (int)(r / (unsigned)a.Tl) * a.Xb + xl;
        g.b = (g.t + g.x + g.y + a.parity) & 1;
        s = (((long)g.t * a.X + g.x) * a.Y + g.y) * a.Zh + g.zh;
    }
    const size_t vh = (size_t)a.vh;
    const size_t pb = vh * 16; // plane bytes
    const char *in = (const char *)a.in;
    const char *lk_own = (const char *)a.links + (size_t)(a.parity * 4) * LB * vh;       // links based at output parity
    const char *lk_nbr = (const char *)a.links + (size_t)((1 - a.parity) * 4) * LB * vh; // links based at input parity

    uint64_t pol_l = 0, pol_s = 0;
    if constexpr (LHINT == LD_STREAM_EF) pol_l = make_policy_evict_first();
    if constexpr (SHINT == LD_KEEP) pol_s = make_policy_evict_last();

    if constexpr (KSPLIT == 1) {
        Real acc[4][2 * D];
#pragma unroll
        for (int al = 0; al < 4; ++al)
#pragma unroll
            for (int c = 0; c < 2 * D; ++c) acc[al][c] = 0;

        auto hop = [&](auto mu_c, auto dir_c) {
            constexpr int MU = decltype(mu_c)::value;
            constexpr int DIR = decltype(dir_c)::value;
            long sn; int sign;
            neighbour<MU, DIR>(a, g, s, sn, sign);
            Real psi[8 * D];
            load_record<SHINT, 8 * D>(psi, in, vh, (size_t)sn, pol_s);
            Real u[LNREAL];
            if constexpr (DIR == 0) load_record<LHINT, LNREAL>(u, lk_own + (size_t)MU * LB * vh, vh, (size_t)s, pol_l);
            else                    load_record<LHINT, LNREAL>(u, lk_nbr + (size_t)MU * LB * vh, vh, (size_t)sn, pol_l);
            constexpr int P0 = (MU == 0 || MU == 3) ? 2 : 3;
            constexpr int P1 = 5 - P0;
            const Real sg = (Real)sign;
            with_link<D, LK, Real>(u, [&](auto lk_c, const Real *ul) {
                constexpr int K = decltype(lk_c)::value;
                if constexpr (PackedHop<K, Real>::value) hop_pair_packed<MU, DIR, D, K>(ul, psi, sg, acc);
                else {
                    hop_component<MU, DIR, D, K, Real>(ul, psi + 0 * 2 * D, psi + P0 * 2 * D, (Real)1, sg, acc[0], acc[P0]);
                    hop_component<MU, DIR, D, K, Real>(ul, psi + 1 * 2 * D, psi + P1 * 2 * D, (Real)(MU >= 2 ? -1 : 1), sg, acc[1], acc[P1]);
                }
            });
        };
        using I0 = std::integral_constant<int, 0>; using I1 = std::integral_constant<int, 1>;
        using I2 = std::integral_constant<int, 2>; using I3 = std::integral_constant<int, 3>;
        hop(I0{}, I0{}); hop(I0{}, I1{});
        hop(I1{}, I0{}); hop(I1{}, I1{});
        hop(I2{}, I0{}); hop(I2{}, I1{});
        hop(I3{}, I0{}); hop(I3{}, I1{});

        Real o[8 * D];
        [[maybe_unused]] Real n2 = 0, dre = 0, dim = 0;
        if constexpr (MASS) {
            const Real be[2] = { coef_beta<Real>(a, 0), coef_beta<Real>(a, 1) };
            Real self[8 * D];
            load_record<LD_STREAM, 8 * D>(self, (const char *)a.self, vh, (size_t)s, 0);
            const Real al_[2] = { coef_alpha<Real>(a, 0), coef_alpha<Real>(a, 1) };
#pragma unroll
            for (int al = 0; al < 4; ++al)
#pragma unroll
                for (int c = 0; c < 2 * D; ++c) o[al * 2 * D + c] = fma(al_[al >> 1], self[al * 2 * D + c], be[al >> 1] * acc[al][c]);
            if constexpr (CLV == 1) site_matvec<Real, D>(o, self, (const char *)a.site_mat, vh, (size_t)s);
            if constexpr (RED) {
#pragma unroll
                for (int e = 0; e < 4 * D; ++e) {
                    const Real sr = self[2 * e], si = self[2 * e + 1], orr = o[2 * e], oi = o[2 * e + 1];
                    n2 = fma(orr, orr, fma(oi, oi, n2));
                    dre = fma(sr, orr, fma(si, oi, dre));   // conj(self) * out
                    dim = fma(sr, oi, fma(-si, orr, dim));
                }
            }
        } else {
#pragma unroll
            for (int al = 0; al < 4; ++al)
#pragma unroll
                for (int c = 0; c < 2 * D; ++c) o[al * 2 * D + c] = (Real)-0.5 * acc[al][c]; // plain Dphi
            if constexpr (CLV == 2) {
                Real hv[8 * D];
#pragma unroll
                for (int e = 0; e < 8 * D; ++e) { hv[e] = o[e]; o[e] = 0; }
                site_matvec<Real, D>(o, hv, (const char *)a.site_mat, vh, (size_t)s);
            }
        }
        if (live) store_planes<STHINT, 8 * D / RPV>((char *)a.out + (size_t)s * 16, pb, o);
        if constexpr (RED) {
            double v[3] = { live ? (double)n2 : 0.0, live ? (double)dre : 0.0, live ? (double)dim : 0.0 };
            if (grid_reduce<3>(v, a.red_partial, a.red_ticket)) { a.red_result[0] = v[0]; a.red_result[1] = v[1]; a.red_result[2] = v[2]; }
        }
    } else {
        // two threads per site: thread k owns h_k.  accK -> out_k, accP -> out_{k+2} (mu = 0,3),
        // accQ -> out_{3-k} (mu = 1,2), exchanged with the partner lane at the end.
        Real accK[2 * D], accP[2 * D], accQ[2 * D];
#pragma unroll
        for (int c = 0; c < 2 * D; ++c) { accK[c] = 0; accP[c] = 0; accQ[c] = 0; }

        auto hop = [&](auto mu_c, auto dir_c) {
            constexpr int MU = decltype(mu_c)::value;
            constexpr int DIR = decltype(dir_c)::value;
            long sn; int sign;
            neighbour<MU, DIR>(a, g, s, sn, sign);
            constexpr bool STRAIGHT = (MU == 0 || MU == 3);
            const int pk = STRAIGHT ? k + 2 : 3 - k;
            Real pa[2 * D], pbv[2 * D];
            const char *base = in + (size_t)sn * 16;
            load_planes<SHINT, SPV>(pa, base + (size_t)(k * SPV) * pb, pb, pol_s);
            load_planes<SHINT, SPV>(pbv, base + (size_t)(pk * SPV) * pb, pb, pol_s);
            Real u[LNREAL];
            if constexpr (DIR == 0) load_record<LHINT, LNREAL>(u, lk_own + (size_t)MU * LB * vh, vh, (size_t)s, pol_l);
            else                    load_record<LHINT, LNREAL>(u, lk_nbr + (size_t)MU * LB * vh, vh, (size_t)sn, pol_l);
            const Real sk = (MU >= 2 && k == 1) ? (Real)-1 : (Real)1;
            with_link<D, LK, Real>(u, [&](auto lk_c, const Real *ul) {
                hop_component<MU, DIR, D, decltype(lk_c)::value, Real>(ul, pa, pbv, sk, (Real)sign, accK, STRAIGHT ? accP : accQ);
            });
        };
        using I0 = std::integral_constant<int, 0>; using I1 = std::integral_constant<int, 1>;
        using I2 = std::integral_constant<int, 2>; using I3 = std::integral_constant<int, 3>;
        hop(I0{}, I0{}); hop(I0{}, I1{});
        hop(I1{}, I0{}); hop(I1{}, I1{});
        hop(I2{}, I0{}); hop(I2{}, I1{});
        hop(I3{}, I0{}); hop(I3{}, I1{});

#pragma unroll
        for (int c = 0; c < 2 * D; ++c) accP[c] += __shfl_xor_sync(0xffffffffu, accQ[c], 1);

        [[maybe_unused]] Real n2 = 0, dre = 0, dim = 0;
        if constexpr (MASS) {
            const Real be[2] = { coef_beta<Real>(a, 0), coef_beta<Real>(a, 1) };
            Real sa[2 * D], sb[2 * D];
            const char *base = (const char *)a.self + (size_t)s * 16;
            load_planes<LD_STREAM, SPV>(sa, base + (size_t)(k * SPV) * pb, pb, 0);
            load_planes<LD_STREAM, SPV>(sb, base + (size_t)((k + 2) * SPV) * pb, pb, 0);
            const Real al_[2] = { coef_alpha<Real>(a, 0), coef_alpha<Real>(a, 1) };
#pragma unroll
            for (int c = 0; c < 2 * D; ++c) {
                accK[c] = fma(al_[0], sa[c], be[0] * accK[c]);   // component k   (upper)
                accP[c] = fma(al_[1], sb[c], be[1] * accP[c]);   // component k+2 (lower)
            }
            if constexpr (RED) {
#pragma unroll
                for (int e = 0; e < D; ++e) {
                    n2 = fma(accK[2 * e], accK[2 * e], fma(accK[2 * e + 1], accK[2 * e + 1], n2));
                    n2 = fma(accP[2 * e], accP[2 * e], fma(accP[2 * e + 1], accP[2 * e + 1], n2));
                    dre = fma(sa[2 * e], accK[2 * e], fma(sa[2 * e + 1], accK[2 * e + 1], dre));
                    dre = fma(sb[2 * e], accP[2 * e], fma(sb[2 * e + 1], accP[2 * e + 1], dre));
                    dim = fma(sa[2 * e], accK[2 * e + 1], fma(-sa[2 * e + 1], accK[2 * e], dim));
                    dim = fma(sb[2 * e], accP[2 * e + 1], fma(-sb[2 * e + 1], accP[2 * e], dim));
                }
            }
        } else {
#pragma unroll
            for (int c = 0; c < 2 * D; ++c) { accK[c] *= (Real)-0.5; accP[c] *= (Real)-0.5; } // plain Dphi
        }
        if (live) {
            char *ob = (char *)a.out + (size_t)s * 16;
            store_planes<STHINT, SPV>(ob + (size_t)(k * SPV) * pb, pb, accK);
            store_planes<STHINT, SPV>(ob + (size_t)((k + 2) * SPV) * pb, pb, accP);
        }
        if constexpr (RED) {
            double v[3] = { live ? (double)n2 : 0.0, live ? (double)dre : 0.0, live ? (double)dim : 0.0 };
            if (grid_reduce<3>(v, a.red_partial, a.red_ticket)) { a.red_result[0] = v[0]; a.red_result[1] = v[1]; a.red_result[2] = v[2]; }
        }
    }
}

} // namespace hr
