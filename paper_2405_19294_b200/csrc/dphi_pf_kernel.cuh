// dphi_pf_kernel.cuh -- Dphi with the NEXT hop's operands in flight while the current hop is computed.
//
// dphi_kernel (one thread per site) loads the neighbour spinor and the link of a hop into registers and
// then runs ~300 dependent FMAs on them; with the 8-16 warps per SM its register budget allows, ncu shows
// the warps waiting on the long scoreboard (memory latency), not on bandwidth.  Here every thread copies
// the operands of hop h+1 with cp.async (LDGSTS) into its own 16-byte slots of a double-buffered shared-
// memory stage while it computes hop h from registers: the loads cost no registers while they are in
// flight, and one more hop's worth of bytes per thread is outstanding.  This is north_star's "TMA or
// shared-memory staging of neighbour spinors" put to the use that pays on B200: latency hiding.  (Re-use
// of neighbour spinors across sites already happens in L1/L2 -- DRAM traffic equals the compulsory bytes,
// profiles/ -- so staging for re-use would gain nothing.)
//
// Slots are private to a thread (slot(v, tid) = ((buf * NSLOT + v) * blockDim.x + tid) * 16): no
// __syncthreads anywhere, cp.async.wait_group only; consecutive threads own consecutive 16-byte slots,
// so both the LDGSTS writes and the LDS reads are bank-conflict free, and the global side of every
// LDGSTS is the same coalesced 512-byte-per-warp plane access as in dphi_kernel.
#pragma once
#include "dphi_kernel.cuh"

namespace hr {

__device__ __forceinline__ void cp_async16_ca(uint32_t dst, const void *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async16_cg(uint32_t dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async8_ca(uint32_t dst, const void *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4_ca(uint32_t dst, const void *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ void lds16(double *d, uint32_t addr)
{
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(d[0]), "=d"(d[1]) : "r"(addr));
}
__device__ __forceinline__ void lds16(float *d, uint32_t addr)
{
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3]) : "r"(addr));
}

template <typename Real, int D, int LK> struct PfGeom {
    static constexpr int RPV = 16 / (int)sizeof(Real);
    static constexpr int LNREAL = LinkGeom<LK, D>::NREAL;
    static constexpr int NVS = 8 * D / RPV;              // spinor vectors
    static constexpr int NVL = LNREAL / RPV;             // full link vectors
    static constexpr int TAIL = LNREAL - NVL * RPV;      // reals in the link's tail plane
    static constexpr int NSLOT = NVS + NVL + (TAIL ? 1 : 0);
    static constexpr size_t smem_bytes(int block) { return (size_t)2 * NSLOT * block * 16; }
};

template <typename Real, int D, int LK, bool MASS, bool RED, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) dphi_pf_kernel(const DphiArgs a)
{
    static_assert(!RED || MASS, "the fused reduction needs the self field");
    using G = PfGeom<Real, D, LK>;
    constexpr int RPV = G::RPV, LNREAL = G::LNREAL, NVS = G::NVS, NVL = G::NVL, TAIL = G::TAIL, NSLOT = G::NSLOT;
    constexpr size_t LB = (size_t)LNREAL * sizeof(Real);
    extern __shared__ __align__(16) char pf_smem[];
    if (a.skip != nullptr && *a.skip != 0) return;

    long s = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = s < a.vh;
    if (!live) s = a.vh - 1;
    SiteGeom g;
    {
        unsigned r = (unsigned)s;
        g.zh = (int)(r % (unsigned)a.Zh); r /= (unsigned)a.Zh;
        g.y = (int)(r % (unsigned)a.Y); r /= (unsigned)a.Y;
        const int xl = (int)(r % (unsigned)a.Xb); r /= (unsigned)a.Xb;
        g.t = (int)(r % (unsigned)a.T);
        g.x = (int)(r / (unsigned)a.T) * a.Xb + xl;
        g.b = (g.t + g.x + g.y + a.parity) & 1;
        s = (((long)g.t * a.X + g.x) * a.Y + g.y) * a.Zh + g.zh;
    }
    const size_t vh = (size_t)a.vh;
    const size_t pb = vh * 16;
    const char *in = (const char *)a.in;
    const char *lk_own = (const char *)a.links + (size_t)(a.parity * 4) * LB * vh;
    const char *lk_nbr = (const char *)a.links + (size_t)((1 - a.parity) * 4) * LB * vh;
    const uint32_t stride = blockDim.x * 16u;                                        // bytes between slots v, v+1
    const uint32_t base0 = (uint32_t)__cvta_generic_to_shared(pf_smem) + threadIdx.x * 16u;
    const uint32_t base1 = base0 + (uint32_t)NSLOT * stride;

    auto issue = [&](auto mu_c, auto dir_c, uint32_t dst) {
        constexpr int MU = decltype(mu_c)::value;
        constexpr int DIR = decltype(dir_c)::value;
        long sn; int sign;
        neighbour<MU, DIR>(a, g, s, sn, sign);
        const char *ps = in + (size_t)sn * 16;
#pragma unroll
        for (int v = 0; v < NVS; ++v) cp_async16_ca(dst + v * stride, ps + v * pb);      // spinors: L1 + L2 (re-used)
        const char *pl = (DIR == 0 ? lk_own : lk_nbr) + (size_t)MU * LB * vh;
        const size_t li = DIR == 0 ? (size_t)s : (size_t)sn;
#pragma unroll
        for (int v = 0; v < NVL; ++v) cp_async16_cg(dst + (NVS + v) * stride, pl + li * 16 + v * pb); // links: past L1
        if constexpr (TAIL != 0) {
            const char *pt = pl + (size_t)NVL * 16 * vh + li * (TAIL * sizeof(Real));
            const uint32_t dt = dst + (NVS + NVL) * stride;
            if constexpr (TAIL * sizeof(Real) == 8) cp_async8_ca(dt, pt);
            else
#pragma unroll
                for (int e = 0; e < TAIL; ++e) cp_async4_ca(dt + 4 * e, pt + 4 * e);
        }
        cp_async_commit();
    };

    Real acc[4][2 * D];
#pragma unroll
    for (int al = 0; al < 4; ++al)
#pragma unroll
        for (int c = 0; c < 2 * D; ++c) acc[al][c] = 0;

    auto hop = [&](auto mu_c, auto dir_c, uint32_t src, auto &&issue_next) {
        constexpr int MU = decltype(mu_c)::value;
        constexpr int DIR = decltype(dir_c)::value;
        cp_async_wait_all();
        Real psi[8 * D];
        Real u[NVL * RPV + (TAIL ? RPV : 0)];
#pragma unroll
        for (int v = 0; v < NVS; ++v) lds16(psi + v * RPV, src + v * stride);
#pragma unroll
        for (int v = 0; v < NVL + (TAIL ? 1 : 0); ++v) lds16(u + v * RPV, src + (NVS + v) * stride);
        issue_next();
        long sn; int sign;
        neighbour<MU, DIR>(a, g, s, sn, sign);
        constexpr int P0 = (MU == 0 || MU == 3) ? 2 : 3;
        constexpr int P1 = 5 - P0;
        const Real sg = (Real)sign;
        with_link<D, LK, Real>(u, [&](auto lk_c, const Real *ul) {
            constexpr int K = decltype(lk_c)::value;
            hop_component<MU, DIR, D, K, Real>(ul, psi + 0 * 2 * D, psi + P0 * 2 * D, (Real)1, sg, acc[0], acc[P0]);
            hop_component<MU, DIR, D, K, Real>(ul, psi + 1 * 2 * D, psi + P1 * 2 * D, (Real)(MU >= 2 ? -1 : 1), sg, acc[1], acc[P1]);
        });
    };
    using I0 = std::integral_constant<int, 0>; using I1 = std::integral_constant<int, 1>;
    using I2 = std::integral_constant<int, 2>; using I3 = std::integral_constant<int, 3>;
    issue(I0{}, I0{}, base0);
    hop(I0{}, I0{}, base0, [&] { issue(I0{}, I1{}, base1); });
    hop(I0{}, I1{}, base1, [&] { issue(I1{}, I0{}, base0); });
    hop(I1{}, I0{}, base0, [&] { issue(I1{}, I1{}, base1); });
    hop(I1{}, I1{}, base1, [&] { issue(I2{}, I0{}, base0); });
    hop(I2{}, I0{}, base0, [&] { issue(I2{}, I1{}, base1); });
    hop(I2{}, I1{}, base1, [&] { issue(I3{}, I0{}, base0); });
    hop(I3{}, I0{}, base0, [&] { issue(I3{}, I1{}, base1); });
    hop(I3{}, I1{}, base1, [] {});

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
