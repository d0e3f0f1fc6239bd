// dphi_cpo_kernel.cuh -- colour-parallel Dphi with the two-index representation applied ON THE FLY from the fundamental
// link (kernel variant 6 for the link kinds LK_SYM_OTF / LK_ASYM_OTF, both halves at once).
//
// With the colour vector written as the (anti)symmetric N x N matrix Psi' (dphi_kernel.cuh: twoindex_mul),
// R(U) psi <-> M' = W Psi' W^T, W = U (forward hop) or U^dagger (backward hop).  One thread per (site, ROW i of M'):
//   * it owns the components (i, j), j >= i (symmetric) or j > i (antisymmetric) -- projects them (four spin components
//     of each of its colours of the neighbour spinor -> two half-spinor entries), exchanges them through shared memory
//     exactly as dphi_cp_kernel does, accumulates and finally stores them;
//   * per hop it reads all h back, forms Psi' in registers, A_l = sum_k W_ik Psi'_kl with ROW i of W, then only the
//     entries M'_ij = sum_l A_l W_jl it owns -- no redundant arithmetic between the N threads of a site;
//   * the fundamental link (N^2 complex, 144 B for SU(3) in fp64) is read through L1 by the N warps of the CTA.
// A thread carries at most N colours x 4 spins of accumulators instead of d_R x 4 (128 registers instead of 254).
// MEASURED: 1.6-2.7x slower than the one-thread-per-site on-the-fly kernel -- the link and Psi' are
// re-read by each of the N threads of a site.  Not a default anywhere; kept as evidence of the design point.
#pragma once
#include "dphi_cp_kernel.cuh"

namespace hr {

template <typename Real, int N, bool SYM> struct CpoGeom {
    static constexpr int D = SYM ? N * (N + 1) / 2 : N * (N - 1) / 2;
    static constexpr int SITES = 32;
    static constexpr int THREADS = SITES * N;
    static constexpr size_t smem_bytes() { return (size_t)4 * 2 * D * SITES * sizeof(CpPair<Real>); }
#ifndef HR_CPO_REGS
#define HR_CPO_REGS 128
#endif
    static constexpr int MINB = 65536 / (THREADS * HR_CPO_REGS) < 1 ? 1 : 65536 / (THREADS * HR_CPO_REGS);
};

template <typename Real, int N, bool SYM, bool MASS, bool RED>
__global__ void __launch_bounds__((CpoGeom<Real, N, SYM>::THREADS), (CpoGeom<Real, N, SYM>::MINB)) dphi_cpo_kernel(const DphiArgs a)
{
    static_assert(!RED || MASS, "the fused reduction needs the self field");
    using G = CpoGeom<Real, N, SYM>;
    constexpr int D = G::D, SITES = G::SITES;
    constexpr int LNREAL = 2 * N * N;
    constexpr size_t LB = (size_t)LNREAL * sizeof(Real);
    constexpr Real SQ2 = (Real)1.4142135623730951, ISQ2 = (Real)0.7071067811865476;
    if (a.skip != nullptr && *a.skip != 0) return;
    extern __shared__ __align__(16) unsigned char cp_smem[];
    CpPair<Real> *hs = reinterpret_cast<CpPair<Real> *>(cp_smem);          // [slot][k][a][site]

    const int sl = (int)threadIdx.x % SITES, row = (int)threadIdx.x / SITES;
    long s = (long)blockIdx.x * SITES + sl;
    const bool live = s < a.vh;
    if (!live) s = a.vh - 1;
    SiteGeom g;
    {
        unsigned r = (unsigned)s;
        g.zh = (int)(r % (unsigned)a.Zh); r /= (unsigned)a.Zh;
        g.y = (int)(r % (unsigned)a.Y); r /= (unsigned)a.Y;
        g.x = (int)(r % (unsigned)a.X);
        g.t = (int)(r / (unsigned)a.X);
        g.b = (g.t + g.x + g.y + a.parity) & 1;
    }
    const size_t vh = (size_t)a.vh;
    const char *in = (const char *)a.in;
    const char *lk_own = (const char *)a.links + (size_t)(a.parity * 4) * LB * vh;
    const char *lk_nbr = (const char *)a.links + (size_t)((1 - a.parity) * 4) * LB * vh;
    // component of the pair (row, j) in the lexicographic pair order of reading C8; owned iff j >= row (sym) / j > row
    const int off = SYM ? row * N - row * (row - 1) / 2 - row : row * (N - 1) - row * (row - 1) / 2 - row - 1; // comp = off + j
    auto owned = [&](int j) { return SYM ? j >= row : j > row; };

    Real acc[N][4][2];
#pragma unroll
    for (int j = 0; j < N; ++j)
#pragma unroll
        for (int al = 0; al < 4; ++al) acc[j][al][0] = acc[j][al][1] = 0;

    auto project = [&](auto mu_c, auto dir_c, int slot, long &sn, int &sign) {
        constexpr int MU = decltype(mu_c)::value;
        constexpr int DIR = decltype(dir_c)::value;
        constexpr int S = DIR ? -1 : 1;
        constexpr int CRE = (MU == 0 || MU == 2) ? S : 0;
        constexpr int CIM = (MU == 0 || MU == 2) ? 0 : S;
        constexpr int P0 = (MU == 0 || MU == 3) ? 2 : 3;
        constexpr int P1 = 5 - P0;
        neighbour<MU, DIR>(a, g, s, sn, sign);
#pragma unroll
        for (int j = 0; j < N; ++j) {
            if (!owned(j)) continue;
            const int c = off + j;
            Real p[4][2];
#pragma unroll
            for (int al = 0; al < 4; ++al) load_cplx<LD_DEFAULT, 8 * D>(p[al][0], p[al][1], in, vh, (size_t)sn, al * D + c, 0);
            CpPair<Real> h0, h1;
            add_c<CRE, CIM>(h0.re, h0.im, p[0][0], p[0][1], p[P0][0], p[P0][1], (Real)1);
            add_c<CRE, CIM>(h1.re, h1.im, p[1][0], p[1][1], p[P1][0], p[P1][1], (Real)(MU >= 2 ? -1 : 1));
            hs[((slot * 2 + 0) * D + c) * SITES + sl] = h0;
            hs[((slot * 2 + 1) * D + c) * SITES + sl] = h1;
        }
    };
    auto multiply = [&](auto mu_c, auto dir_c, int slot, long sn, int sign) {
        constexpr int MU = decltype(mu_c)::value;
        constexpr int DIR = decltype(dir_c)::value;
        constexpr int S = DIR ? -1 : 1;
        constexpr int CRE = (MU == 0 || MU == 2) ? S : 0;
        constexpr int CIM = (MU == 0 || MU == 2) ? 0 : S;
        constexpr int P0 = (MU == 0 || MU == 3) ? 2 : 3;
        constexpr int P1 = 5 - P0;
        const char *lbase = (DIR == 0 ? lk_own : lk_nbr) + (size_t)MU * LB * vh;
        const size_t ls = DIR == 0 ? (size_t)s : (size_t)sn;
        // W = U (forward) or U^dagger (backward): the full matrix (compile-time indices) and my row (runtime index)
        Real u[2 * N * N], wrow[2 * N];
#pragma unroll
        for (int e = 0; e < N * N; ++e) load_cplx<LD_DEFAULT, LNREAL>(u[2 * e], u[2 * e + 1], lbase, vh, ls, e, 0);
#pragma unroll
        for (int k = 0; k < N; ++k) {
            load_cplx<LD_DEFAULT, LNREAL>(wrow[2 * k], wrow[2 * k + 1], lbase, vh, ls, DIR == 0 ? row * N + k : k * N + row, 0);
            if constexpr (DIR == 1) wrow[2 * k + 1] = -wrow[2 * k + 1];
        }
        auto wr = [&](int j, int l) -> Real { return DIR == 1 ? u[2 * (l * N + j)] : u[2 * (j * N + l)]; };
        auto wi = [&](int j, int l) -> Real { return DIR == 1 ? -u[2 * (l * N + j) + 1] : u[2 * (j * N + l) + 1]; };
        const Real sg = (Real)sign;
        const Real sk1 = (Real)(MU >= 2 ? -1 : 1);
#pragma unroll
        for (int kk = 0; kk < 2; ++kk) {                                   // the two half-spinor components
            // Psi' (dphi_kernel.cuh: off-diagonal entries are the components, diagonal ones sqrt2 h (sym) or 0)
            Real pr[N][N], pi[N][N];
            {
                int c = 0;
#pragma unroll
                for (int i = 0; i < N; ++i)
#pragma unroll
                    for (int j = i; j < N; ++j) {
                        if (i == j && !SYM) { pr[i][i] = 0; pi[i][i] = 0; continue; }
                        const CpPair<Real> h = hs[((slot * 2 + kk) * D + c) * SITES + sl];
                        ++c;
                        if (i == j) { pr[i][i] = SQ2 * h.re; pi[i][i] = SQ2 * h.im; }
                        else {
                            pr[i][j] = h.re; pi[i][j] = h.im;
                            pr[j][i] = SYM ? h.re : -h.re; pi[j][i] = SYM ? h.im : -h.im;
                        }
                    }
            }
            // A_l = sum_k W_{row,k} Psi'_{k,l}
            Real ar[N], ai[N];
#pragma unroll
            for (int l = 0; l < N; ++l) {
                Real re = 0, im = 0;
#pragma unroll
                for (int k = 0; k < N; ++k) {
                    if (!SYM && k == l) continue;
                    re = fma(wrow[2 * k], pr[k][l], re); re = fma(-wrow[2 * k + 1], pi[k][l], re);
                    im = fma(wrow[2 * k], pi[k][l], im); im = fma(wrow[2 * k + 1], pr[k][l], im);
                }
                ar[l] = re; ai[l] = im;
            }
            // M'_{row,j} = sum_l A_l W_{j,l}, owned entries only; chi = M' (off-diagonal) or M' / sqrt2 (diagonal)
#pragma unroll
            for (int j = 0; j < N; ++j) {
                if (!owned(j)) continue;
                Real re = 0, im = 0;
#pragma unroll
                for (int l = 0; l < N; ++l) {
                    re = fma(ar[l], wr(j, l), re); re = fma(-ai[l], wi(j, l), re);
                    im = fma(ar[l], wi(j, l), im); im = fma(ai[l], wr(j, l), im);
                }
                if (SYM && j == row) { re *= ISQ2; im *= ISQ2; }
                const Real w = kk == 0 ? sg : sg * sk1;
                acc[j][kk][0] = fma(sg, re, acc[j][kk][0]);
                acc[j][kk][1] = fma(sg, im, acc[j][kk][1]);
                constexpr int PK0 = P0, PK1 = P1;
                if (kk == 0) acc_conj_c<CRE, CIM>(acc[j][PK0][0], acc[j][PK0][1], re, im, w);
                else acc_conj_c<CRE, CIM>(acc[j][PK1][0], acc[j][PK1][1], re, im, w);
            }
        }
    };
    using I0 = std::integral_constant<int, 0>; using I1 = std::integral_constant<int, 1>;
    using I2 = std::integral_constant<int, 2>; using I3 = std::integral_constant<int, 3>;
    long sn[4]; int sign[4];
    project(I0{}, I0{}, 0, sn[0], sign[0]); project(I0{}, I1{}, 1, sn[1], sign[1]);
    project(I1{}, I0{}, 2, sn[2], sign[2]); project(I1{}, I1{}, 3, sn[3], sign[3]);
    __syncthreads();
    multiply(I0{}, I0{}, 0, sn[0], sign[0]); multiply(I0{}, I1{}, 1, sn[1], sign[1]);
    multiply(I1{}, I0{}, 2, sn[2], sign[2]); multiply(I1{}, I1{}, 3, sn[3], sign[3]);
    __syncthreads();
    project(I2{}, I0{}, 0, sn[0], sign[0]); project(I2{}, I1{}, 1, sn[1], sign[1]);
    project(I3{}, I0{}, 2, sn[2], sign[2]); project(I3{}, I1{}, 3, sn[3], sign[3]);
    __syncthreads();
    multiply(I2{}, I0{}, 0, sn[0], sign[0]); multiply(I2{}, I1{}, 1, sn[1], sign[1]);
    multiply(I3{}, I0{}, 2, sn[2], sign[2]); multiply(I3{}, I1{}, 3, sn[3], sign[3]);

    [[maybe_unused]] Real n2 = 0, dre = 0, dim = 0;
#pragma unroll
    for (int j = 0; j < N; ++j) {
        if (!owned(j)) continue;
        const int c = off + j;
#pragma unroll
        for (int al = 0; al < 4; ++al) {
            Real orr, oi;
            if constexpr (MASS) {
                Real sr, si;
                load_cplx<LD_STREAM, 8 * D>(sr, si, (const char *)a.self, vh, (size_t)s, al * D + c, 0);
                const Real alc = coef_alpha<Real>(a, al >> 1), bec = coef_beta<Real>(a, al >> 1);
                orr = fma(alc, sr, bec * acc[j][al][0]);
                oi = fma(alc, si, bec * acc[j][al][1]);
                if constexpr (RED) {
                    n2 = fma(orr, orr, fma(oi, oi, n2));
                    dre = fma(sr, orr, fma(si, oi, dre));
                    dim = fma(sr, oi, fma(-si, orr, dim));
                }
            } else {
                orr = (Real)-0.5 * acc[j][al][0];
                oi = (Real)-0.5 * acc[j][al][1];
            }
            if (live) {
                const int e = al * D + c;
                if constexpr (sizeof(Real) == 8)
                    *reinterpret_cast<double2 *>((char *)a.out + ((size_t)e * vh + (size_t)s) * 16) = make_double2((double)orr, (double)oi);
                else
                    *reinterpret_cast<float2 *>((char *)a.out + ((size_t)(e >> 1) * vh + (size_t)s) * 16 + (size_t)(e & 1) * 8) =
                        make_float2((float)orr, (float)oi);
            }
        }
    }
    if constexpr (RED) {
        double v[3] = { live ? (double)n2 : 0.0, live ? (double)dre : 0.0, live ? (double)dim : 0.0 };
        if (grid_reduce<3>(v, a.red_partial, a.red_ticket)) { a.red_result[0] = v[0]; a.red_result[1] = v[1]; a.red_result[2] = v[2]; }
    }
}

template <typename Real, int D, int LK, bool MASS, bool RED>
static hr_status launch_cpo(const DphiArgs &a, cudaStream_t st)
{
    static_assert(LK == LK_SYM_OTF || LK == LK_ASYM_OTF, "on-the-fly colour-parallel kernel: two-index representations");
    constexpr int N = LinkGeom<LK, D>::N;
    using G = CpoGeom<Real, N, LK == LK_SYM_OTF>;
    static_assert(G::D == D, "representation dimension");
    static_assert(G::smem_bytes() <= 48 * 1024, "static shared-memory budget");
    const long grid = (a.vh + G::SITES - 1) / G::SITES;
    if (RED && (unsigned long)grid > kRedMaxBlocks) { set_error("fused Dphi reduction: too many CTAs"); return HR_EUNSUPPORTED; }
    dphi_cpo_kernel<Real, N, LK == LK_SYM_OTF, MASS, RED><<<(unsigned)grid, G::THREADS, G::smem_bytes(), st>>>(a);
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { set_error("dphi on-the-fly colour kernel launch failed: %s", cudaGetErrorString(e)); return HR_ECUDA; }
    return HR_OK;
}

} // namespace hr
