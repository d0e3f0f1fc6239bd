// dphi_loop_kernel.cuh -- the one-thread-per-site Dphi kernel with the four directions as a REAL loop: kernel variant 11
// `site_loop`.
//
// dphi_kernel.cuh unrolls all eight hops with compile-time projector tables; for a site with much arithmetic (the
// two-index representations applied on the fly: 230 FMA per half-spinor component and hop) that is 4800-6500 SASS
// instructions = 77-105 KB of straight-line code that every warp streams through once.  ncu on the fp32 on-the-fly
// sextet: issue slots 51-58 % busy with 0.7-0.9 warps per issue stalled on `no_instruction` -- instruction fetch
// (profiles/r2_otf_ncu.md).  Here the body holds ONE direction (a forward and a backward hop, DIR stays compile-time
// because U and U^dagger multiply differently) and runs four times with the projector as run-time data:
//   h_k = psi_k + c_k psi_{p(k)},   c_0 = s (1 or i),  c_1 = s sk (1 or i),  s = +1 forward / -1 backward,
//   p(0) = 2 (mu = 0, 3) or 3 (mu = 1, 2),  sk = -1 for mu >= 2;
// the partner component is picked by its ADDRESS (a run-time plane offset), the lower accumulators by two selects.
// Code size / 4; 24 extra FMA and 24 selects per hop.  Needs vector-aligned spin components (2 d_R reals a whole
// number of 16-byte vectors).  Same epilogue as dphi_kernel (self term, fused reduction, skip flag); no fused site matrix.
#pragma once
#include "dphi_kernel.cuh"

namespace hr {

// one hop with run-time projector: (cre, cim) = c_0 / s,  sk1 = sign of component 1,  straight = (p(0) == 2)
template <int DIR, int D, int LK, typename Real>
__device__ __forceinline__ void loop_hop(const Real *u, const Real *a0, const Real *b0, const Real *a1, const Real *b1,
                                         Real cre, Real cim, Real sk1, Real sgn, bool straight, Real (&acc)[4][2 * D])
{
    constexpr Real S = DIR ? (Real)-1 : (Real)1;
    const Real c0r = S * cre, c0i = S * cim, c1r = c0r * sk1, c1i = c0i * sk1;
    Real h0[2 * D], h1[2 * D], chi0[2 * D], chi1[2 * D];
#pragma unroll
    for (int c = 0; c < D; ++c) {
        // h = a + (cr + i ci) b
        h0[2 * c] = fma(c0r, b0[2 * c], fma(-c0i, b0[2 * c + 1], a0[2 * c]));
        h0[2 * c + 1] = fma(c0r, b0[2 * c + 1], fma(c0i, b0[2 * c], a0[2 * c + 1]));
        h1[2 * c] = fma(c1r, b1[2 * c], fma(-c1i, b1[2 * c + 1], a1[2 * c]));
        h1[2 * c + 1] = fma(c1r, b1[2 * c + 1], fma(c1i, b1[2 * c], a1[2 * c + 1]));
    }
    with_link<D, LK, Real>(u, [&](auto lk_c, const Real *ul) {
        constexpr int K = decltype(lk_c)::value;
        link_mul<D, K, DIR == 1>(chi0, ul, h0);
        link_mul<D, K, DIR == 1>(chi1, ul, h1);
    });
    // out_k += sgn chi_k;  out_{p(k)} += sgn conj(c_k) chi_k
    const Real w0r = sgn * c0r, w0i = sgn * c0i, w1r = sgn * c1r, w1i = sgn * c1i;
#pragma unroll
    for (int c = 0; c < D; ++c) {
        acc[0][2 * c] = fma(sgn, chi0[2 * c], acc[0][2 * c]);
        acc[0][2 * c + 1] = fma(sgn, chi0[2 * c + 1], acc[0][2 * c + 1]);
        acc[1][2 * c] = fma(sgn, chi1[2 * c], acc[1][2 * c]);
        acc[1][2 * c + 1] = fma(sgn, chi1[2 * c + 1], acc[1][2 * c + 1]);
        // x = conj(w) chi = (wr - i wi)(xr + i xi)
        const Real x0r = fma(w0r, chi0[2 * c], w0i * chi0[2 * c + 1]), x0i = fma(w0r, chi0[2 * c + 1], -w0i * chi0[2 * c]);
        const Real x1r = fma(w1r, chi1[2 * c], w1i * chi1[2 * c + 1]), x1i = fma(w1r, chi1[2 * c + 1], -w1i * chi1[2 * c]);
        acc[2][2 * c] += straight ? x0r : x1r;
        acc[2][2 * c + 1] += straight ? x0i : x1i;
        acc[3][2 * c] += straight ? x1r : x0r;
        acc[3][2 * c + 1] += straight ? x1i : x0i;
    }
}

template <typename Real, int D, int LK, bool MASS, bool RED, int LHINT, int SHINT, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) dphi_loop_kernel(const DphiArgs a)
{
    static_assert(!RED || MASS, "the fused reduction needs the self field");
    if (a.skip != nullptr && *a.skip != 0) return;
    constexpr int LNREAL = LinkGeom<LK, D>::NREAL;
    constexpr int RPV = 16 / (int)sizeof(Real);
    constexpr int SPV = 2 * D / RPV;
    static_assert((2 * D) % RPV == 0, "site_loop needs vector-aligned spin components");
    constexpr size_t LB = (size_t)LNREAL * sizeof(Real);

    long s = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = s < a.vh;
    if (!live) s = a.vh - 1;
    int ct, cx, cy, zh, b;
    {
        unsigned r = (unsigned)s;
        zh = (int)(r % (unsigned)a.Zh); r /= (unsigned)a.Zh;
        cy = (int)(r % (unsigned)a.Y); r /= (unsigned)a.Y;
        const int xl = (int)(r % (unsigned)a.Xb); r /= (unsigned)a.Xb;
        ct = (int)(r % (unsigned)a.T);
        cx = (int)(r / (unsigned)a.T) * a.Xb + xl;
        b = (ct + cx + cy + a.parity) & 1;
        s = (((long)ct * a.X + cx) * a.Y + cy) * a.Zh + zh;
    }
    const size_t vh = (size_t)a.vh;
    const size_t pb = vh * 16;
    const char *in = (const char *)a.in;
    const char *lk_own = (const char *)a.links + (size_t)(a.parity * 4) * LB * vh;
    const char *lk_nbr = (const char *)a.links + (size_t)((1 - a.parity) * 4) * LB * vh;
    uint64_t pol_l = 0, pol_s = 0;
    if constexpr (LHINT == LD_STREAM_EF) pol_l = make_policy_evict_first();
    if constexpr (SHINT == LD_KEEP) pol_s = make_policy_evict_last();

    Real acc[4][2 * D];
#pragma unroll
    for (int al = 0; al < 4; ++al)
#pragma unroll
        for (int c = 0; c < 2 * D; ++c) acc[al][c] = 0;

#pragma unroll 1
    for (int mu = 0; mu < 4; ++mu) {
        const bool straight = mu == 0 || mu == 3;
        const int p0 = straight ? 2 : 3, p1 = 5 - p0;
        const Real cre = (mu & 1) ? (Real)0 : (Real)1, cim = (mu & 1) ? (Real)1 : (Real)0;
        const Real sk1 = mu >= 2 ? (Real)-1 : (Real)1;
        // neighbours of direction mu: half indices and seam signs
        long sf, sb_;
        int sgf = 1, sgb = 1;
        if (mu < 3) {
            const int coord = mu == 0 ? ct : mu == 1 ? cx : cy;
            const int ext = mu == 0 ? a.T : mu == 1 ? a.X : a.Y;
            const long st = mu == 0 ? (long)a.X * a.Y * a.Zh : mu == 1 ? (long)a.Y * a.Zh : (long)a.Zh;
            const bool wf = coord == ext - 1, wb = coord == 0;
            sf = wf ? s - (ext - 1) * st : s + st;
            sb_ = wb ? s + (ext - 1) * st : s - st;
            sgf = wf ? a.bc[mu] : 1;
            sgb = wb ? a.bc[mu] : 1;
        } else {
            const bool wf = zh == a.Zh - 1, wb = zh == 0;
            sf = b ? (wf ? s - (a.Zh - 1) : s + 1) : s;
            sb_ = b ? s : (wb ? s + (a.Zh - 1) : s - 1);
            sgf = (b && wf) ? a.bc[3] : 1;
            sgb = (!b && wb) ? a.bc[3] : 1;
        }
        auto hop = [&](auto dir_c, long sn, int sign) {
            constexpr int DIR = decltype(dir_c)::value;
            const char *sp = in + (size_t)sn * 16;
            Real a0[2 * D], b0[2 * D], a1[2 * D], b1[2 * D];
            load_planes<SHINT, SPV>(a0, sp, pb, pol_s);
            load_planes<SHINT, SPV>(a1, sp + (size_t)SPV * pb, pb, pol_s);
            load_planes<SHINT, SPV>(b0, sp + (size_t)(p0 * SPV) * pb, pb, pol_s);
            load_planes<SHINT, SPV>(b1, sp + (size_t)(p1 * SPV) * pb, pb, pol_s);
            Real u[LNREAL];
            if constexpr (DIR == 0) load_record<LHINT, LNREAL>(u, lk_own + (size_t)mu * LB * vh, vh, (size_t)s, pol_l);
            else                    load_record<LHINT, LNREAL>(u, lk_nbr + (size_t)mu * LB * vh, vh, (size_t)sn, pol_l);
            loop_hop<DIR, D, LK, Real>(u, a0, b0, a1, b1, cre, cim, sk1, (Real)sign, straight, acc);
        };
        hop(std::integral_constant<int, 0>{}, sf, sgf);
        hop(std::integral_constant<int, 1>{}, sb_, sgb);
    }

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
        if constexpr (RED) {
#pragma unroll
            for (int e = 0; e < 4 * D; ++e) {
                const Real sr = self[2 * e], si = self[2 * e + 1], orr = o[2 * e], oi = o[2 * e + 1];
                n2 = fma(orr, orr, fma(oi, oi, n2));
                dre = fma(sr, orr, fma(si, oi, dre));
                dim = fma(sr, oi, fma(-si, orr, dim));
            }
        }
    } else {
#pragma unroll
        for (int al = 0; al < 4; ++al)
#pragma unroll
            for (int c = 0; c < 2 * D; ++c) o[al * 2 * D + c] = (Real)-0.5 * acc[al][c];
    }
    if (live) store_planes<ST_DEFAULT, 8 * D / RPV>((char *)a.out + (size_t)s * 16, pb, o);
    if constexpr (RED) {
        double v[3] = { live ? (double)n2 : 0.0, live ? (double)dre : 0.0, live ? (double)dim : 0.0 };
        if (grid_reduce<3>(v, a.red_partial, a.red_ticket)) { a.red_result[0] = v[0]; a.red_result[1] = v[1]; a.red_result[2] = v[2]; }
    }
}

} // namespace hr
