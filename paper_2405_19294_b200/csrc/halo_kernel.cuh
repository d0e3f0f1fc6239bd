// halo_kernel.cuh -- SURVEY.md section 8(e)/(f) NEXT-2: Dphi_eo on a lattice split into slabs along t
// (one slab per GPU), with the paper's half-spinor exchange ("partially applying the Dirac
// operator before the synchronization to the send buffer ... it is only necessary to send a half-spinor").
//
// A rank owns T_l consecutive time-slices.  For output parity p its Dphi_eo needs, beyond its own sites,
//   * at its slice t = 0      the backward hop  (1+gamma_0) U_0(x-0)^dagger psi(x-0):  site AND link belong to the
//     PREVIOUS rank, which therefore sends  chi = U_0(y)^dagger P+ psi(y)  for y in its LAST slice ("up" message);
//   * at its slice t = T_l-1  the forward hop   (1-gamma_0) U_0(x) psi(x+0):  the link is its own, so the NEXT rank
//     sends only  h = P- psi(y)  for y in its FIRST slice ("down" message).
// P-+ psi = (psi_0 +- psi_2, psi_1 +- psi_3) in the chiral basis of reading C1 (table in dphi_kernel.cuh), so a
// message is 2 d_R complex per face site -- half a spinor; links are never exchanged.
//
//   halo_pack_kernel   one thread per face site: writes both messages (send buffers may be PEER memory mapped over
//                      NVLink: the projection is then fused with the transfer, plain coalesced 16-byte stores).
//   (interior)         the ordinary dphi_kernel on the local slab with bc[0] = 0: hops across the slab boundary
//                      contribute nothing; runs while the messages travel.
//   halo_apply_kernel  one thread per face site: out(t=0) += beta s_prev R+(chi_recv), out(t=T_l-1) += beta s_next
//                      R-(U_0(x) h_recv); s = bc[0] on the global seam (rank 0's first / last rank's last slice).
// Face buffers use the plane layout of hr_internal.h: [16-byte vector v][face site f], f = (x*Y + y)*Zh + zh.
#pragma once
#include "dphi_kernel.cuh"

namespace hr {


template <typename Real, int D, int LK>
__global__ void __launch_bounds__(128) halo_pack_kernel(const HaloArgs a)
{
    constexpr int LNREAL = LinkGeom<LK, D>::NREAL;
    constexpr int RPV = 16 / (int)sizeof(Real);
    constexpr size_t LB = (size_t)LNREAL * sizeof(Real);
    const long f = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= a.nface) return;
    const size_t vh = (size_t)a.vh, nf = (size_t)a.nface;
    const char *in = (const char *)a.in;
    // down message: first slice, h = (psi0 + psi2, psi1 + psi3)
    {
        Real psi[8 * D], h[4 * D];
        load_record<LD_DEFAULT, 8 * D>(psi, in, vh, (size_t)f, 0);
#pragma unroll
        for (int c = 0; c < 2 * D; ++c) { h[c] = psi[c] + psi[4 * D + c]; h[2 * D + c] = psi[2 * D + c] + psi[6 * D + c]; }
        store_planes<ST_DEFAULT, 4 * D / RPV>((char *)a.send_dn + (size_t)f * 16, nf * 16, h);
    }
    // up message: last slice, chi = U_0(y)^dagger (psi0 - psi2, psi1 - psi3); U_0(y) is based at the INPUT parity
    {
        const size_t sy = (size_t)(a.Tl - 1) * nf + (size_t)f;
        Real psi[8 * D], u[LNREAL], h0[2 * D], h1[2 * D], c0[2 * D], c1[2 * D], chi[4 * D];
        load_record<LD_DEFAULT, 8 * D>(psi, in, vh, sy, 0);
        load_record<LD_STREAM, LNREAL>(u, (const char *)a.links + (size_t)((1 - a.parity) * 4) * LB * vh, vh, sy, 0);
#pragma unroll
        for (int c = 0; c < 2 * D; ++c) { h0[c] = psi[c] - psi[4 * D + c]; h1[c] = psi[2 * D + c] - psi[6 * D + c]; }
        link_mul<D, LK, true>(c0, u, h0);
        link_mul<D, LK, true>(c1, u, h1);
#pragma unroll
        for (int c = 0; c < 2 * D; ++c) { chi[c] = c0[c]; chi[2 * D + c] = c1[c]; }
        store_planes<ST_DEFAULT, 4 * D / RPV>((char *)a.send_up + (size_t)f * 16, nf * 16, chi);
    }
}

template <typename Real, int D, int LK>
__global__ void __launch_bounds__(128) halo_apply_kernel(const HaloArgs a)
{
    constexpr int LNREAL = LinkGeom<LK, D>::NREAL;
    constexpr int RPV = 16 / (int)sizeof(Real);
    constexpr size_t LB = (size_t)LNREAL * sizeof(Real);
    const long f = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= a.nface) return;
    const size_t vh = (size_t)a.vh, nf = (size_t)a.nface;
    Real be[2];
    if constexpr (sizeof(Real) == 8) { be[0] = (Real)a.beta[0]; be[1] = (Real)a.beta[1]; }
    else { be[0] = a.betaf[0]; be[1] = a.betaf[1]; }
    char *out = (char *)a.out;
    // slice 0: backward hop from the previous rank, (1+gamma_0) chi = (chi0, chi1, -chi0, -chi1)
    {
        Real chi[4 * D], o[8 * D];
        load_planes<LD_STREAM, 4 * D / RPV>(chi, (const char *)a.recv_prev + (size_t)f * 16, nf * 16, 0);
        load_record<LD_DEFAULT, 8 * D>(o, out, vh, (size_t)f, 0);
        const Real s0 = be[0] * (Real)a.sign_prev, s1 = be[1] * (Real)a.sign_prev;
#pragma unroll
        for (int c = 0; c < 4 * D; ++c) { o[c] = fma(s0, chi[c], o[c]); o[4 * D + c] = fma(-s1, chi[c], o[4 * D + c]); }
        store_planes<ST_DEFAULT, 8 * D / RPV>(out + (size_t)f * 16, vh * 16, o);
    }
    // slice T_l-1: forward hop to the next rank, (1-gamma_0) U_0(x) h = (chi0, chi1, chi0, chi1), own link
    {
        const size_t sx = (size_t)(a.Tl - 1) * nf + (size_t)f;
        Real h[4 * D], u[LNREAL], h0[2 * D], h1[2 * D], c0[2 * D], c1[2 * D], o[8 * D];
        load_planes<LD_STREAM, 4 * D / RPV>(h, (const char *)a.recv_next + (size_t)f * 16, nf * 16, 0);
        load_record<LD_STREAM, LNREAL>(u, (const char *)a.links + (size_t)(a.parity * 4) * LB * vh, vh, sx, 0);
        load_record<LD_DEFAULT, 8 * D>(o, out, vh, sx, 0);
#pragma unroll
        for (int c = 0; c < 2 * D; ++c) { h0[c] = h[c]; h1[c] = h[2 * D + c]; }
        link_mul<D, LK, false>(c0, u, h0);
        link_mul<D, LK, false>(c1, u, h1);
        const Real s0 = be[0] * (Real)a.sign_next, s1 = be[1] * (Real)a.sign_next;
#pragma unroll
        for (int c = 0; c < 2 * D; ++c) {
            o[c] = fma(s0, c0[c], o[c]);
            o[2 * D + c] = fma(s0, c1[c], o[2 * D + c]);
            o[4 * D + c] = fma(s1, c0[c], o[4 * D + c]);
            o[6 * D + c] = fma(s1, c1[c], o[6 * D + c]);
        }
        store_planes<ST_DEFAULT, 8 * D / RPV>(out + sx * 16, vh * 16, o);
    }
}

} // namespace hr
