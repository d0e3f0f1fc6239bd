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
// Face buffers use the plane layout of hr_internal.h: [16-byte vector v][face site f].
//
// 4-D block decomposition: the same two kernels for every direction MU.  With the projector table of dphi_kernel.cuh
// (h_k = psi_k + sk_k c psi_{p(k)}, c = +c0 forward / -c0 backward, c0 = 1 (mu = 0,2) or i (mu = 1,3)):
//   "down" message (to the previous rank in MU): h = P^-_mu psi of my FIRST slice x_mu = 0 (forward projector);
//   "up" message (to the next rank in MU): chi = U_mu(y)^dagger P^+_mu psi of my LAST slice x_mu = L_mu - 1.
// Face sites of direction MU are enumerated as f = the half index with the coordinate x_mu dropped (mu = 0,1,2: one site
// per (other coordinates, zh)); for mu = 3 the face z = 0 holds the sites with offset bit b = 0 and the face z = Z-1 those
// with b = 1, one per (t, x, y/2), y's parity fixed by the site parity -- sender and receiver enumerate them alike.
#pragma once
#include "dphi_kernel.cuh"

namespace hr {

// half index of face site f of direction MU on the first (side 0) or last (side 1) slice, for sites of parity `par`
template <int MU> __device__ __forceinline__ size_t face_site(const HaloArgs &a, int par, int side, long f)
{
    const unsigned X = (unsigned)a.X, Y = (unsigned)a.Y, Zh = (unsigned)a.Zh;
    unsigned r = (unsigned)f;
    if constexpr (MU == 0) {
        return (size_t)f + (side ? (size_t)(a.T - 1) * X * Y * Zh : 0);
    } else if constexpr (MU == 1) {
        const unsigned zh = r % Zh; r /= Zh;
        const unsigned y = r % Y, t = r / Y, x = side ? X - 1 : 0;
        return (((size_t)t * X + x) * Y + y) * Zh + zh;
    } else if constexpr (MU == 2) {
        const unsigned zh = r % Zh; r /= Zh;
        const unsigned x = r % X, t = r / X, y = side ? Y - 1 : 0;
        return (((size_t)t * X + x) * Y + y) * Zh + zh;
    } else {
        const unsigned Yh = Y / 2;
        const unsigned yh = r % Yh; r /= Yh;
        const unsigned x = r % X, t = r / X;
        const unsigned y = 2 * yh + ((t + x + (unsigned)par + (unsigned)side) & 1u);   // offset bit b = side
        return (((size_t)t * X + x) * Y + y) * Zh + (side ? Zh - 1 : 0);
    }
}

template <int MU> struct HopTable {
    static constexpr int CRE = (MU == 0 || MU == 2) ? 1 : 0;   // c0
    static constexpr int CIM = (MU == 0 || MU == 2) ? 0 : 1;
    static constexpr int P0 = (MU == 0 || MU == 3) ? 2 : 3;
    static constexpr int P1 = 5 - P0;
};

// both messages of face site f of direction MU
template <typename Real, int D, int LK, int MU>
__device__ __forceinline__ void halo_pack_site(const HaloArgs &a, long f)
{
    constexpr int LNREAL = LinkGeom<LK, D>::NREAL;
    constexpr int RPV = 16 / (int)sizeof(Real);
    constexpr size_t LB = (size_t)LNREAL * sizeof(Real);
    using H = HopTable<MU>;
    if (f >= a.nface) return;
    const size_t vh = (size_t)a.vh, nf = (size_t)a.nface;
    const char *in = (const char *)a.in;
    const int q = 1 - a.parity;                         // parity of the input sites
    const Real sk1 = (Real)(MU >= 2 ? -1 : 1);
    // down message: first slice, forward projector h_k = psi_k + sk_k c0 psi_{p(k)}
    {
        const size_t sy = face_site<MU>(a, q, 0, f);
        Real psi[8 * D], h[4 * D];
        load_record<LD_DEFAULT, 8 * D>(psi, in, vh, sy, 0);
#pragma unroll
        for (int c = 0; c < D; ++c) {
            add_c<H::CRE, H::CIM>(h[2 * c], h[2 * c + 1], psi[2 * c], psi[2 * c + 1], psi[H::P0 * 2 * D + 2 * c], psi[H::P0 * 2 * D + 2 * c + 1], (Real)1);
            add_c<H::CRE, H::CIM>(h[2 * D + 2 * c], h[2 * D + 2 * c + 1], psi[2 * D + 2 * c], psi[2 * D + 2 * c + 1],
                                  psi[H::P1 * 2 * D + 2 * c], psi[H::P1 * 2 * D + 2 * c + 1], sk1);
        }
        store_planes<ST_DEFAULT, 4 * D / RPV>((char *)a.send_dn + (size_t)f * 16, nf * 16, h);
    }
    // up message: last slice, chi = U_mu(y)^dagger (psi_k - sk_k c0 psi_{p(k)}); U_mu(y) is based at the INPUT parity
    {
        const size_t sy = face_site<MU>(a, q, 1, f);
        Real psi[8 * D], u[LNREAL], h0[2 * D], h1[2 * D], c0[2 * D], c1[2 * D], chi[4 * D];
        load_record<LD_DEFAULT, 8 * D>(psi, in, vh, sy, 0);
        load_record<LD_STREAM, LNREAL>(u, (const char *)a.links + (size_t)(q * 4 + MU) * LB * vh, vh, sy, 0);
#pragma unroll
        for (int c = 0; c < D; ++c) {
            add_c<-H::CRE, -H::CIM>(h0[2 * c], h0[2 * c + 1], psi[2 * c], psi[2 * c + 1], psi[H::P0 * 2 * D + 2 * c], psi[H::P0 * 2 * D + 2 * c + 1], (Real)1);
            add_c<-H::CRE, -H::CIM>(h1[2 * c], h1[2 * c + 1], psi[2 * D + 2 * c], psi[2 * D + 2 * c + 1],
                                    psi[H::P1 * 2 * D + 2 * c], psi[H::P1 * 2 * D + 2 * c + 1], sk1);
        }
        link_mul<D, LK, true>(c0, u, h0);
        link_mul<D, LK, true>(c1, u, h1);
#pragma unroll
        for (int c = 0; c < 2 * D; ++c) { chi[c] = c0[c]; chi[2 * D + c] = c1[c]; }
        store_planes<ST_DEFAULT, 4 * D / RPV>((char *)a.send_up + (size_t)f * 16, nf * 16, chi);
    }
}

template <typename Real, int D, int LK, int MU>
__global__ void __launch_bounds__(128) halo_pack_kernel(const HaloArgs a)
{
    halo_pack_site<Real, D, LK, MU>(a, (long)blockIdx.x * blockDim.x + threadIdx.x);
}

// the faces of ALL split directions in one launch (a 4-D block decomposition packs up to four directions from the same
// input field: four launches of 7-40 us each were launch-bound).  The CTAs of direction
// k are [first[k], first[k+1]): a CTA never straddles two directions, the switch is uniform.
struct HaloMultiArgs {
    HaloArgs a[4];
    unsigned first[5];
    int mu[4];
    int ndir;
    int slot[4];   // direction mu -> its entry of a[], -1 if mu is not split (fused apply)
};
template <typename Real, int D, int LK>
__global__ void __launch_bounds__(128) halo_pack_multi_kernel(const __grid_constant__ HaloMultiArgs g)
{
    int k = 0;
    while (k + 1 < g.ndir && blockIdx.x >= g.first[k + 1]) ++k;
    const long f = (long)(blockIdx.x - g.first[k]) * blockDim.x + threadIdx.x;
    switch (g.mu[k]) {
    case 0: halo_pack_site<Real, D, LK, 0>(g.a[k], f); break;
    case 1: halo_pack_site<Real, D, LK, 1>(g.a[k], f); break;
    case 2: halo_pack_site<Real, D, LK, 2>(g.a[k], f); break;
    default: halo_pack_site<Real, D, LK, 3>(g.a[k], f); break;
    }
}

// The two face terms of direction MU, added to the site's spinor o[] held in registers (shared by the per-direction and the
// fused apply kernels, so that both perform the same sequence of roundings):
//   apply_prev  first slice: backward hop from the previous rank; reconstruct with c = -c0:
//               out_k += chi_k, out_{p(k)} += sk_k conj(-c0) chi_k
//   apply_next  last slice: forward hop to the next rank, chi = U_mu(x) h_recv with the OWN link; reconstruct with c = +c0
template <typename Real, int D, int LK, int MU>
__device__ __forceinline__ void apply_prev(Real (&o)[8 * D], const HaloArgs &a, size_t f, const Real (&be)[2])
{
    constexpr int RPV = 16 / (int)sizeof(Real);
    using H = HopTable<MU>;
    const Real sk1 = (Real)(MU >= 2 ? -1 : 1);
    Real chi[4 * D];
    load_planes<LD_STREAM, 4 * D / RPV>(chi, (const char *)a.recv_prev + f * 16, (size_t)a.nface * 16, 0);
    const Real s0 = be[0] * (Real)a.sign_prev, s1 = be[1] * (Real)a.sign_prev;
#pragma unroll
    for (int c = 0; c < D; ++c) {
        o[2 * c] = fma(s0, chi[2 * c], o[2 * c]);
        o[2 * c + 1] = fma(s0, chi[2 * c + 1], o[2 * c + 1]);
        o[2 * D + 2 * c] = fma(s0, chi[2 * D + 2 * c], o[2 * D + 2 * c]);
        o[2 * D + 2 * c + 1] = fma(s0, chi[2 * D + 2 * c + 1], o[2 * D + 2 * c + 1]);
        acc_conj_c<-H::CRE, -H::CIM>(o[H::P0 * 2 * D + 2 * c], o[H::P0 * 2 * D + 2 * c + 1], chi[2 * c], chi[2 * c + 1], s1);
        acc_conj_c<-H::CRE, -H::CIM>(o[H::P1 * 2 * D + 2 * c], o[H::P1 * 2 * D + 2 * c + 1], chi[2 * D + 2 * c], chi[2 * D + 2 * c + 1], s1 * sk1);
    }
}
template <typename Real, int D, int LK, int MU>
__device__ __forceinline__ void apply_next(Real (&o)[8 * D], const HaloArgs &a, size_t f, size_t sx, const Real (&be)[2])
{
    constexpr int LNREAL = LinkGeom<LK, D>::NREAL;
    constexpr int RPV = 16 / (int)sizeof(Real);
    constexpr size_t LB = (size_t)LNREAL * sizeof(Real);
    using H = HopTable<MU>;
    const Real sk1 = (Real)(MU >= 2 ? -1 : 1);
    const size_t vh = (size_t)a.vh;
    Real h[4 * D], u[LNREAL], h0[2 * D], h1[2 * D], c0[2 * D], c1[2 * D];
    load_planes<LD_STREAM, 4 * D / RPV>(h, (const char *)a.recv_next + f * 16, (size_t)a.nface * 16, 0);
    load_record<LD_STREAM, LNREAL>(u, (const char *)a.links + (size_t)(a.parity * 4 + MU) * LB * vh, vh, sx, 0);
#pragma unroll
    for (int c = 0; c < 2 * D; ++c) { h0[c] = h[c]; h1[c] = h[2 * D + c]; }
    link_mul<D, LK, false>(c0, u, h0);
    link_mul<D, LK, false>(c1, u, h1);
    const Real s0 = be[0] * (Real)a.sign_next, s1 = be[1] * (Real)a.sign_next;
#pragma unroll
    for (int c = 0; c < D; ++c) {
        o[2 * c] = fma(s0, c0[2 * c], o[2 * c]);
        o[2 * c + 1] = fma(s0, c0[2 * c + 1], o[2 * c + 1]);
        o[2 * D + 2 * c] = fma(s0, c1[2 * c], o[2 * D + 2 * c]);
        o[2 * D + 2 * c + 1] = fma(s0, c1[2 * c + 1], o[2 * D + 2 * c + 1]);
        acc_conj_c<H::CRE, H::CIM>(o[H::P0 * 2 * D + 2 * c], o[H::P0 * 2 * D + 2 * c + 1], c0[2 * c], c0[2 * c + 1], s1);
        acc_conj_c<H::CRE, H::CIM>(o[H::P1 * 2 * D + 2 * c], o[H::P1 * 2 * D + 2 * c + 1], c1[2 * c], c1[2 * c + 1], s1 * sk1);
    }
}

template <typename Real> __device__ __forceinline__ void halo_beta(Real (&be)[2], const HaloArgs &a)
{
    if constexpr (sizeof(Real) == 8) { be[0] = (Real)a.beta[0]; be[1] = (Real)a.beta[1]; }
    else { be[0] = a.betaf[0]; be[1] = a.betaf[1]; }
}

template <typename Real, int D, int LK, int MU>
__global__ void __launch_bounds__(128) halo_apply_kernel(const HaloArgs a)
{
    constexpr int RPV = 16 / (int)sizeof(Real);
    const long f = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= a.nface) return;
    const size_t vh = (size_t)a.vh;
    Real be[2];
    halo_beta(be, a);
    char *out = (char *)a.out;
    {
        const size_t sx = face_site<MU>(a, a.parity, 0, f);
        Real o[8 * D];
        load_record<LD_DEFAULT, 8 * D>(o, out, vh, sx, 0);
        apply_prev<Real, D, LK, MU>(o, a, (size_t)f, be);
        store_planes<ST_DEFAULT, 8 * D / RPV>(out + sx * 16, vh * 16, o);
    }
    {
        const size_t sx = face_site<MU>(a, a.parity, 1, f);
        Real o[8 * D];
        load_record<LD_DEFAULT, 8 * D>(o, out, vh, sx, 0);
        apply_next<Real, D, LK, MU>(o, a, (size_t)f, sx, be);
        store_planes<ST_DEFAULT, 8 * D / RPV>(out + sx * 16, vh * 16, o);
    }
}

// The face terms of ALL split directions in one launch.  A site on an edge or corner of the block receives a term from each
// of its faces, and out += term is not associative: to stay bitwise equal to the per-direction launches (ascending mu, each
// a read-modify-write of out) every boundary site is updated by exactly ONE thread, which adds the terms of all its faces in
// ascending mu with the spinor in registers.  Threads are laid out as in halo_pack_multi_kernel -- thread (k, f) visits the
// two sites f of the first and last slice of direction mu_k -- and thread (k, f) OWNS a site iff the site lies on no face of
// a split direction below mu_k; the others skip it.  Face index of a site in direction mu = the inverse of face_site.
template <typename Real, int D, int LK, int MU>
__device__ __forceinline__ void apply_dir(Real (&o)[8 * D], const HaloMultiArgs &g, int t, int x, int y, int zh, int b, size_t sx,
                                          const Real (&be)[2])
{
    const int slot = g.slot[MU];
    if (slot < 0) return;
    const HaloArgs &a = g.a[slot];
    bool lo, hi;
    size_t f;
    if constexpr (MU == 0) { lo = t == 0; hi = t == a.T - 1; f = ((size_t)x * a.Y + y) * a.Zh + zh; }
    else if constexpr (MU == 1) { lo = x == 0; hi = x == a.X - 1; f = ((size_t)t * a.Y + y) * a.Zh + zh; }
    else if constexpr (MU == 2) { lo = y == 0; hi = y == a.Y - 1; f = ((size_t)t * a.X + x) * a.Zh + zh; }
    else { lo = zh == 0 && b == 0; hi = zh == a.Zh - 1 && b == 1; f = ((size_t)t * a.X + x) * (a.Y / 2) + y / 2; }
    if (lo) apply_prev<Real, D, LK, MU>(o, a, f, be);
    if (hi) apply_next<Real, D, LK, MU>(o, a, f, sx, be);
}

template <typename Real, int D, int LK>
__global__ void __launch_bounds__(128) halo_apply_multi_kernel(const __grid_constant__ HaloMultiArgs g)
{
    constexpr int RPV = 16 / (int)sizeof(Real);
    int k = 0;
    while (k + 1 < g.ndir && blockIdx.x >= g.first[k + 1]) ++k;
    const HaloArgs &a = g.a[k];
    const long f = (long)(blockIdx.x - g.first[k]) * blockDim.x + threadIdx.x;
    if (f >= a.nface) return;
    const int mu = g.mu[k];
    const size_t vh = (size_t)a.vh;
    Real be[2];
    halo_beta(be, a);
    char *out = (char *)a.out;
#pragma unroll 1
    for (int side = 0; side < 2; ++side) {
        const size_t sx = mu == 0 ? face_site<0>(a, a.parity, side, f) : mu == 1 ? face_site<1>(a, a.parity, side, f)
                        : mu == 2 ? face_site<2>(a, a.parity, side, f) : face_site<3>(a, a.parity, side, f);
        unsigned r = (unsigned)sx;
        const int zh = (int)(r % (unsigned)a.Zh); r /= (unsigned)a.Zh;
        const int y = (int)(r % (unsigned)a.Y); r /= (unsigned)a.Y;
        const int x = (int)(r % (unsigned)a.X);
        const int t = (int)(r / (unsigned)a.X);
        const int b = (t + x + y + a.parity) & 1;
        // owner: no face of a split direction below mu holds this site
        bool mine = true;
        if (mu > 0 && g.slot[0] >= 0 && (t == 0 || t == a.T - 1)) mine = false;
        if (mu > 1 && g.slot[1] >= 0 && (x == 0 || x == a.X - 1)) mine = false;
        if (mu > 2 && g.slot[2] >= 0 && (y == 0 || y == a.Y - 1)) mine = false;
        if (!mine) continue;
        Real o[8 * D];
        load_record<LD_DEFAULT, 8 * D>(o, out, vh, sx, 0);
        apply_dir<Real, D, LK, 0>(o, g, t, x, y, zh, b, sx, be);
        apply_dir<Real, D, LK, 1>(o, g, t, x, y, zh, b, sx, be);
        apply_dir<Real, D, LK, 2>(o, g, t, x, y, zh, b, sx, be);
        apply_dir<Real, D, LK, 3>(o, g, t, x, y, zh, b, sx, be);
        store_planes<ST_DEFAULT, 8 * D / RPV>(out + sx * 16, vh * 16, o);
    }
}

} // namespace hr
