// dphi_bulk_kernel.cuh -- Dphi_eo with the operands of every hop staged in shared memory by bulk asynchronous copies
// (TMA, cp.async.bulk + mbarrier), kernel variant 7 `bulk`.
//
// north_star: "TMA or shared-memory staging of neighbour spinors along the fastest lattice direction so they are reused
// across sites".  What the one-thread-per-site kernel (dphi_kernel.cuh) cannot do is keep enough bytes in flight once a
// site's live state fills the register file (registers limit occupancy, bandwidth drops): its loads live
// in registers, 8 warps per SM.  Here the bytes in flight live in shared memory instead:
//
//  * a TILE is R consecutive z-rows (R | Y, n = R * Zh <= 128 sites) of one (t, x): in the [plane][site] layout of
//    hr_internal.h the neighbour spinors and links a tile needs for one hop are, per 16-byte plane, ONE contiguous run
//    of n * 16 bytes (two runs where the y-hop wraps) -- the 1-D bulk-copy case.  The z neighbours of an even-odd
//    compacted row are the same row shifted by 0 / +-1 with the wrap inside the row, so they are in the run as well.
//  * a CTA is persistent (grid = SMs x CTAs per SM) and walks tiles in the x-blocked order of dphi_kernel.cuh.  Warp 0
//    is the PRODUCER: for every (tile, hop) one elected lane waits for a free stage of a ring in shared memory, arms the
//    stage's mbarrier with the byte count and issues ONE tensor-map copy (cp.async.bulk.tensor) for the spinor box
//    [planes][n sites] and one for the link box (+ a 1-D bulk copy for a link's sub-vector tail plane).  (One 1-D
//    copy per plane was measured first: 21-60 UBLKCP per hop, serialised over the lanes at ~80 cycles each, left the
//    producer as the bottleneck at 0.4-0.6 of peak.)  The other warps
//    are CONSUMERS, one thread per site: wait for the stage, read spinor and link with conflict-free 16-byte LDS,
//    release the stage, then project / multiply / accumulate exactly as dphi_kernel does (hop_component is shared).
//    The ring runs across tile boundaries, so there is no ramp or tail per tile and the producer runs up to NSTAGE
//    hops (up to ~200 KB per SM) ahead of the arithmetic.
//  * boundaries by index arithmetic as before: the producer picks the wrapped run, the consumer applies the seam sign.
//
// Same epilogue as dphi_kernel (alpha/beta, gamma5 sign pattern, fused reduction, skip flag); the fused site matrix
// (CLV) is not carried here.
#pragma once
#include <cuda.h>   // CUtensorMap (an opaque 128-byte descriptor; encoded on the host in tma_maps.cu)

#include "dphi_kernel.cuh"

namespace hr {

struct BulkArgs {
    int R;            // rows per tile (divides Y)
    int n;            // sites per tile = R * Zh
    int nstage;       // ring depth
    int tiles_y;      // Y / R
    long ntiles;      // T * X * tiles_y
    unsigned stage_bytes;
};

// tensor maps over the input spinor (sp) and the gauge field (lk): box of [0] a whole tile (n sites), [1] one row
// (Zh sites), [2] a tile less one row -- the last two serve the tiles whose y-hop wraps (two runs per plane)
struct BulkMaps {
    CUtensorMap sp[3];
    CUtensorMap lk[3];
};

hr_status encode_plane_map(void *map64, const void *base, size_t vh, int nplanes, int nfields, size_t field_stride, int box_sites);

__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
// global -> shared bulk copy (TMA, 1-D); completion is signalled on `bar` as `bytes` of transaction count
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// global -> shared tile copies through a tensor map: all planes of `box` consecutive sites starting at 8-byte word c0
__device__ __forceinline__ void tma_2d(uint32_t dst, const CUtensorMap *m, int c0, uint32_t bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(dst), "l"(m), "r"(c0), "r"(0), "r"(bar) : "memory");
}
__device__ __forceinline__ void tma_3d(uint32_t dst, const CUtensorMap *m, int c0, int field, uint32_t bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(dst), "l"(m), "r"(c0), "r"(0), "r"(field), "r"(bar) : "memory");
}

__device__ __forceinline__ void lds_vec(double *d, const unsigned char *p)
{
    const double2 v = *reinterpret_cast<const double2 *>(p);
    d[0] = v.x; d[1] = v.y;
}
__device__ __forceinline__ void lds_vec(float *d, const unsigned char *p)
{
    const float4 v = *reinterpret_cast<const float4 *>(p);
    d[0] = v.x; d[1] = v.y; d[2] = v.z; d[3] = v.w;
}

__host__ __device__ constexpr unsigned bulk_r128(unsigned x) { return (x + 127u) & ~127u; }

template <typename Real, int D, int LK> struct BulkGeom {
    static constexpr int RPV = 16 / (int)sizeof(Real);
    static constexpr int LNREAL = LinkGeom<LK, D>::NREAL;
    static constexpr int NVS = 8 * D / RPV;                  // spinor planes
    static constexpr int NVL = LNREAL / RPV;                 // whole link planes
    static constexpr int LTAIL = LNREAL - NVL * RPV;         // reals in the link's tail plane
    static constexpr int TAILB = LTAIL * (int)sizeof(Real);  // tail bytes per site
    static constexpr int SITE_BYTES = (NVS + NVL) * 16 + TAILB;
    static constexpr int MAXN = 128;                         // consumer threads per CTA (and 2 * MAXN = the TMA box limit)
    static constexpr int MAXT = 32 + MAXN;
    // a stage: [spinor boxes][link boxes][link tails]; each box region has 128 bytes of slack for the second box of a
    // tile whose y-hop wraps (TMA destinations are 128-byte aligned)
    __host__ __device__ static constexpr unsigned sp_region(int n) { return bulk_r128((unsigned)(n * NVS * 16)) + 128u; }
    __host__ __device__ static constexpr unsigned lk_region(int n) { return bulk_r128((unsigned)(n * NVL * 16)) + 128u; }
    __host__ __device__ static constexpr unsigned stage_bytes(int n)
    {
        return bulk_r128(sp_region(n) + lk_region(n) + (((unsigned)(n * TAILB) + 15u) & ~15u));
    }
};

// KS = 1: one consumer thread per site.  KS = 2: two per site, thread k owns half-spinor component k of every hop (the
// pair structure of dphi_kernel: no redundant spinor reads, both lanes read the same link vectors from shared memory --
// a broadcast --, one shuffle at the end): half the live state per thread and twice the warps, for the sites whose
// arithmetic (on-the-fly representations, d_R >= 6) is too much for four warps per SM.
// KS = 2 tiles stop at 112 sites = 7 consumer warps + the producer warp = 8 warps, two per SM sub-partition, each with up to
// 255 registers.  A 128-site tile would be 9 warps: three of them share one sub-partition's 16384 registers, i.e. at most 170
// per thread (this is why ptxas budgets __launch_bounds__(288) like 384 threads; with __maxnreg__(224) instead the launch
// fails with "too many resources requested") -- and at 168 registers these kernels spill.
template <typename Real, int D, int LK, bool MASS, bool RED, int KS>
#ifndef HR_BULK2_MINB
#define HR_BULK2_MINB 1
#endif
__global__ void __launch_bounds__((KS == 1 ? 32 + BulkGeom<Real, D, LK>::MAXN : 256), (KS == 1 ? 1 : HR_BULK2_MINB))
dphi_bulk_kernel(const DphiArgs a, const BulkArgs g, const __grid_constant__ BulkMaps maps)
{
    static_assert(KS == 1 || (2 * D) % (16 / (int)sizeof(Real)) == 0, "two threads per site need vector-aligned spin components");
    using G = BulkGeom<Real, D, LK>;
    constexpr int RPV = G::RPV, LNREAL = G::LNREAL, NVS = G::NVS, NVL = G::NVL, LTAIL = G::LTAIL;
    constexpr int SPV = 2 * D / RPV;                       // planes per spin component (if a component is whole vectors)
    constexpr bool SPLIT_OK = (2 * D) % RPV == 0;          // spin components start on plane boundaries
    constexpr bool EARLY = !SPLIT_OK || D <= 4;            // small sites: read the whole stage, release, then compute
    extern __shared__ __align__(128) unsigned char smem[];
    if (a.skip != nullptr && *a.skip != 0) return;

    const int n = g.n, nstage = g.nstage, Zh = a.Zh, R = g.R;
    const unsigned spr = G::sp_region(n), lkr = G::lk_region(n);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + (size_t)nstage * g.stage_bytes);
    const uint32_t full0 = smem_addr(bars), empty0 = smem_addr(bars + nstage);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ncw = (int)(blockDim.x >> 5) - 1;              // consumer warps
    if (threadIdx.x == 0) {
        for (int k = 0; k < nstage; ++k) { mbar_init(full0 + 8 * k, 1); mbar_init(empty0 + 8 * k, (uint32_t)ncw); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    const size_t vh = (size_t)a.vh;
    const size_t pb = vh * 16;
    constexpr size_t LB = (size_t)LNREAL * sizeof(Real);
    const long rowst = Zh, st_x = (long)a.Y * Zh, st_t = (long)a.X * a.Y * Zh;

    auto decode = [&](long tile, int &t, int &x, int &y0) {
        unsigned r = (unsigned)tile;
        const int yb = (int)(r % (unsigned)g.tiles_y); r /= (unsigned)g.tiles_y;
        const int xl = (int)(r % (unsigned)a.Xb); r /= (unsigned)a.Xb;
        t = (int)(r % (unsigned)a.T);
        x = (int)(r / (unsigned)a.T) * a.Xb + xl;
        y0 = yb * R;
    };

    int stage = 0;
    uint32_t phase = 0;
    auto advance = [&]() { if (++stage == nstage) { stage = 0; phase ^= 1u; } };

    [[maybe_unused]] Real n2 = 0, dre = 0, dim = 0;

    if (warp == 0) {
        // =============================== producer: one elected lane issues the TMA copies ===============================
        if (lane == 0) {
            const uint32_t tx_bytes = (uint32_t)n * (uint32_t)G::SITE_BYTES;
            const char *tail0 = (const char *)a.links + (size_t)NVL * 16 * vh;      // tail plane of link field 0
            for (long tile = blockIdx.x; tile < g.ntiles; tile += gridDim.x) {
                int t, x, y0;
                decode(tile, t, x, y0);
                const long s0 = (((long)t * a.X + x) * a.Y + y0) * Zh;
#pragma unroll 1
                for (int h = 0; h < 8; ++h) {
                    const int mu = h >> 1, dir = h & 1;
                    // neighbour run(s) of this hop in site units: (src, cnt) x up to 2, in consumer order
                    long src0 = s0, src1 = 0;
                    int cnt0 = n, cnt1 = 0;
                    if (mu == 0) {
                        const int tn = dir == 0 ? (t == a.T - 1 ? 0 : t + 1) : (t == 0 ? a.T - 1 : t - 1);
                        src0 = s0 + (long)(tn - t) * st_t;
                    } else if (mu == 1) {
                        const int xn = dir == 0 ? (x == a.X - 1 ? 0 : x + 1) : (x == 0 ? a.X - 1 : x - 1);
                        src0 = s0 + (long)(xn - x) * st_x;
                    } else if (mu == 2) {
                        if (dir == 0) {
                            if (y0 + R < a.Y) src0 = s0 + rowst;
                            else if (R == 1) src0 = s0 - (long)y0 * rowst;               // the single row wraps to y = 0
                            else { src0 = s0 + rowst; cnt0 = n - Zh; src1 = s0 - (long)y0 * rowst; cnt1 = Zh; }
                        } else {
                            if (y0 > 0) src0 = s0 - rowst;
                            else if (R == 1) src0 = s0 + (long)(a.Y - 1) * rowst;        // ... to y = Y-1
                            else { src0 = s0 + (long)(a.Y - 1) * rowst; cnt0 = Zh; src1 = s0; cnt1 = n - Zh; }
                        }
                    }
                    mbar_wait(empty0 + 8 * stage, phase ^ 1u);
                    const uint32_t fb = full0 + 8 * stage;
                    mbar_arrive_expect_tx(fb, tx_bytes);
                    const uint32_t sbase = smem_addr(smem + (size_t)stage * g.stage_bytes);
                    // spinor
                    if (cnt1 == 0) tma_2d(sbase, &maps.sp[0], (int)(2 * src0), fb);
                    else {
                        const int m0 = cnt0 == Zh ? 1 : 2, m1 = 3 - m0;
                        tma_2d(sbase, &maps.sp[m0], (int)(2 * src0), fb);
                        tma_2d(sbase + bulk_r128((unsigned)(NVS * cnt0 * 16)), &maps.sp[m1], (int)(2 * src1), fb);
                    }
                    // link: the forward hop reads the tile's own links, the backward hop the neighbours'
                    const int field = (dir == 0 ? a.parity : 1 - a.parity) * 4 + mu;
                    const uint32_t lbase = sbase + spr;
                    const bool split = dir == 1 && cnt1 != 0;
                    if (!split) tma_3d(lbase, &maps.lk[0], (int)(2 * (dir == 0 ? s0 : src0)), field, fb);
                    else {
                        const int m0 = cnt0 == Zh ? 1 : 2, m1 = 3 - m0;
                        tma_3d(lbase, &maps.lk[m0], (int)(2 * src0), field, fb);
                        tma_3d(lbase + bulk_r128((unsigned)(NVL * cnt0 * 16)), &maps.lk[m1], (int)(2 * src1), field, fb);
                    }
                    if constexpr (LTAIL > 0) {                                          // tail plane: flat [n], 1-D copies
                        const char *tf = tail0 + (size_t)field * LB * vh;
                        const uint32_t tb = lbase + lkr;
                        if (!split) bulk_g2s(tb, tf + (size_t)(dir == 0 ? s0 : src0) * G::TAILB, (uint32_t)(n * G::TAILB), fb);
                        else {
                            bulk_g2s(tb, tf + (size_t)src0 * G::TAILB, (uint32_t)(cnt0 * G::TAILB), fb);
                            bulk_g2s(tb + (uint32_t)(cnt0 * G::TAILB), tf + (size_t)src1 * G::TAILB, (uint32_t)(cnt1 * G::TAILB), fb);
                        }
                    }
                    advance();
                }
            }
        }
    } else {
        // =============================== consumers: one thread per site of the tile ===============================
        const int ic = ((int)threadIdx.x - 32) / KS;
        [[maybe_unused]] const int kk = ((int)threadIdx.x - 32) % KS;   // KS = 2: my half-spinor component
        const bool mine = ic < n;
        const int i = mine ? ic : n - 1;                      // idle lanes shadow the last site (no stores)
        const int row = i / Zh, zh = i - row * Zh;
        const unsigned cC = (unsigned)(n - Zh);               // sites of a tile less one row

        for (long tile = blockIdx.x; tile < g.ntiles; tile += gridDim.x) {
            int t, x, y0;
            decode(tile, t, x, y0);
            const int y = y0 + row;
            const int b = (t + x + y + a.parity) & 1;
            const size_t s = (size_t)((((long)t * a.X + x) * a.Y + y0) * Zh + i);

            if constexpr (KS == 2) {
            // two threads per site: accK -> out_k, accP -> out_{k+2} (mu = 0,3), accQ -> out_{3-k} (mu = 1,2), exchanged with
            // the partner lane at the end (as dphi_kernel's pair branch)
            Real accK[2 * D], accP[2 * D], accQ[2 * D];
#pragma unroll
            for (int c = 0; c < 2 * D; ++c) { accK[c] = 0; accP[c] = 0; accQ[c] = 0; }
            auto hop = [&](auto mu_c, auto dir_c) {
                constexpr int MU = decltype(mu_c)::value;
                constexpr int DIR = decltype(dir_c)::value;
                int j = i, sign = 1;
                // byte offset of this thread's vector in plane 0 and plane stride, for the spinor and the link boxes
                unsigned sp_off, sp_str = (unsigned)n * 16u, lk_off, lk_str = (unsigned)n * 16u;
                if constexpr (MU == 0) sign = (DIR == 0 ? t == a.T - 1 : t == 0) ? a.bc[0] : 1;
                else if constexpr (MU == 1) sign = (DIR == 0 ? x == a.X - 1 : x == 0) ? a.bc[1] : 1;
                else if constexpr (MU == 2) sign = (DIR == 0 ? y == a.Y - 1 : y == 0) ? a.bc[2] : 1;
                else {
                    if constexpr (DIR == 0) {
                        const bool w = zh == Zh - 1;
                        j = b ? (w ? i - (Zh - 1) : i + 1) : i;
                        sign = (b && w) ? a.bc[3] : 1;
                    } else {
                        const bool w = zh == 0;
                        j = b ? i : (w ? i + (Zh - 1) : i - 1);
                        sign = (!b && w) ? a.bc[3] : 1;
                    }
                }
                sp_off = (unsigned)j * 16u;
                lk_off = (unsigned)(DIR == 0 ? i : j) * 16u;
                if constexpr (MU == 2) {
                    if (R > 1) {
                        if constexpr (DIR == 0) {
                            if (y0 + R == a.Y) {                  // boxes: [tile less its last row][row y = 0]
                                if (row < R - 1) sp_str = cC * 16u;
                                else { sp_off = bulk_r128((unsigned)NVS * cC * 16u) + ((unsigned)i - cC) * 16u; sp_str = (unsigned)Zh * 16u; }
                            }
                        } else {
                            if (y0 == 0) {                       // boxes: [row y = Y-1][tile less its first row]
                                if (row == 0) { sp_str = lk_str = (unsigned)Zh * 16u; }
                                else {
                                    sp_off = bulk_r128((unsigned)(NVS * Zh) * 16u) + (unsigned)(i - Zh) * 16u; sp_str = cC * 16u;
                                    lk_off = bulk_r128((unsigned)(NVL * Zh) * 16u) + (unsigned)(i - Zh) * 16u; lk_str = cC * 16u;
                                }
                            }
                        }
                    }
                }
                [[maybe_unused]] const int jl = DIR == 0 ? i : j;
                [[maybe_unused]] constexpr int P0 = (MU == 0 || MU == 3) ? 2 : 3;
                [[maybe_unused]] constexpr int P1 = 5 - P0;
                const Real sgn = (Real)sign;
                constexpr bool STRAIGHT = (MU == 0 || MU == 3);
                const int pk = STRAIGHT ? kk + 2 : 3 - kk;
                mbar_wait(full0 + 8 * stage, phase);
                const unsigned char *sb = smem + (size_t)stage * g.stage_bytes;
                const unsigned char *sp = sb + sp_off;
                const unsigned char *lp = sb + spr + lk_off;
                Real u[LNREAL];
#pragma unroll
                for (int v = 0; v < NVL; ++v) lds_vec(u + v * RPV, lp + (size_t)v * lk_str);
                if constexpr (LTAIL > 0) {
                    const Real *tp = reinterpret_cast<const Real *>(sb + spr + lkr) + (size_t)jl * LTAIL;
#pragma unroll
                    for (int e = 0; e < LTAIL; ++e) u[NVL * RPV + e] = tp[e];
                }
                Real pa[2 * D], pq[2 * D];
#pragma unroll
                for (int v = 0; v < SPV; ++v) {
                    lds_vec(pa + v * RPV, sp + (size_t)(kk * SPV + v) * sp_str);
                    lds_vec(pq + v * RPV, sp + (size_t)(pk * SPV + v) * sp_str);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(empty0 + 8 * stage);
                const Real sk = (MU >= 2 && kk == 1) ? (Real)-1 : (Real)1;
                with_link<D, LK, Real>(u, [&](auto lk_c, const Real *ul) {
                    hop_component<MU, DIR, D, decltype(lk_c)::value, Real>(ul, pa, pq, sk, sgn, accK, STRAIGHT ? accP : accQ);
                });
                advance();
            };
            using I0 = std::integral_constant<int, 0>; using I1 = std::integral_constant<int, 1>;
            using I2 = std::integral_constant<int, 2>; using I3 = std::integral_constant<int, 3>;
            hop(I0{}, I0{}); hop(I0{}, I1{});
            hop(I1{}, I0{}); hop(I1{}, I1{});
            hop(I2{}, I0{}); hop(I2{}, I1{});
            hop(I3{}, I0{}); hop(I3{}, I1{});
#pragma unroll
            for (int c = 0; c < 2 * D; ++c) accP[c] += __shfl_xor_sync(0xffffffffu, accQ[c], 1);
            if constexpr (MASS) {
                const Real be[2] = { coef_beta<Real>(a, 0), coef_beta<Real>(a, 1) };
                Real sa[2 * D], sbv[2 * D];
                const char *base = (const char *)a.self + s * 16;
                load_planes<LD_STREAM, SPV>(sa, base + (size_t)(kk * SPV) * pb, pb, 0);
                load_planes<LD_STREAM, SPV>(sbv, base + (size_t)((kk + 2) * SPV) * pb, pb, 0);
                const Real al_[2] = { coef_alpha<Real>(a, 0), coef_alpha<Real>(a, 1) };
#pragma unroll
                for (int c = 0; c < 2 * D; ++c) {
                    accK[c] = fma(al_[0], sa[c], be[0] * accK[c]);
                    accP[c] = fma(al_[1], sbv[c], be[1] * accP[c]);
                }
                if constexpr (RED) {
                    if (mine) {
#pragma unroll
                        for (int e = 0; e < D; ++e) {
                            n2 = fma(accK[2 * e], accK[2 * e], fma(accK[2 * e + 1], accK[2 * e + 1], n2));
                            n2 = fma(accP[2 * e], accP[2 * e], fma(accP[2 * e + 1], accP[2 * e + 1], n2));
                            dre = fma(sa[2 * e], accK[2 * e], fma(sa[2 * e + 1], accK[2 * e + 1], dre));
                            dre = fma(sbv[2 * e], accP[2 * e], fma(sbv[2 * e + 1], accP[2 * e + 1], dre));
                            dim = fma(sa[2 * e], accK[2 * e + 1], fma(-sa[2 * e + 1], accK[2 * e], dim));
                            dim = fma(sbv[2 * e], accP[2 * e + 1], fma(-sbv[2 * e + 1], accP[2 * e], dim));
                        }
                    }
                }
            } else {
#pragma unroll
                for (int c = 0; c < 2 * D; ++c) { accK[c] *= (Real)-0.5; accP[c] *= (Real)-0.5; }
            }
            if (mine) {
                char *ob = (char *)a.out + s * 16;
                store_planes<ST_DEFAULT, SPV>(ob + (size_t)(kk * SPV) * pb, pb, accK);
                store_planes<ST_DEFAULT, SPV>(ob + (size_t)((kk + 2) * SPV) * pb, pb, accP);
            }
            } else {
            Real acc[4][2 * D];
#pragma unroll
            for (int al = 0; al < 4; ++al)
#pragma unroll
                for (int c = 0; c < 2 * D; ++c) acc[al][c] = 0;

            auto hop = [&](auto mu_c, auto dir_c) {
                constexpr int MU = decltype(mu_c)::value;
                constexpr int DIR = decltype(dir_c)::value;
                int j = i, sign = 1;
                // byte offset of this thread's vector in plane 0 and plane stride, for the spinor and the link boxes
                unsigned sp_off, sp_str = (unsigned)n * 16u, lk_off, lk_str = (unsigned)n * 16u;
                if constexpr (MU == 0) sign = (DIR == 0 ? t == a.T - 1 : t == 0) ? a.bc[0] : 1;
                else if constexpr (MU == 1) sign = (DIR == 0 ? x == a.X - 1 : x == 0) ? a.bc[1] : 1;
                else if constexpr (MU == 2) sign = (DIR == 0 ? y == a.Y - 1 : y == 0) ? a.bc[2] : 1;
                else {
                    if constexpr (DIR == 0) {
                        const bool w = zh == Zh - 1;
                        j = b ? (w ? i - (Zh - 1) : i + 1) : i;
                        sign = (b && w) ? a.bc[3] : 1;
                    } else {
                        const bool w = zh == 0;
                        j = b ? i : (w ? i + (Zh - 1) : i - 1);
                        sign = (!b && w) ? a.bc[3] : 1;
                    }
                }
                sp_off = (unsigned)j * 16u;
                lk_off = (unsigned)(DIR == 0 ? i : j) * 16u;
                if constexpr (MU == 2) {
                    if (R > 1) {
                        if constexpr (DIR == 0) {
                            if (y0 + R == a.Y) {                  // boxes: [tile less its last row][row y = 0]
                                if (row < R - 1) sp_str = cC * 16u;
                                else { sp_off = bulk_r128((unsigned)NVS * cC * 16u) + ((unsigned)i - cC) * 16u; sp_str = (unsigned)Zh * 16u; }
                            }
                        } else {
                            if (y0 == 0) {                       // boxes: [row y = Y-1][tile less its first row]
                                if (row == 0) { sp_str = lk_str = (unsigned)Zh * 16u; }
                                else {
                                    sp_off = bulk_r128((unsigned)(NVS * Zh) * 16u) + (unsigned)(i - Zh) * 16u; sp_str = cC * 16u;
                                    lk_off = bulk_r128((unsigned)(NVL * Zh) * 16u) + (unsigned)(i - Zh) * 16u; lk_str = cC * 16u;
                                }
                            }
                        }
                    }
                }
                [[maybe_unused]] const int jl = DIR == 0 ? i : j;
                [[maybe_unused]] constexpr int P0 = (MU == 0 || MU == 3) ? 2 : 3;
                [[maybe_unused]] constexpr int P1 = 5 - P0;
                const Real sgn = (Real)sign;

                mbar_wait(full0 + 8 * stage, phase);
                const unsigned char *sb = smem + (size_t)stage * g.stage_bytes;
                const unsigned char *sp = sb + sp_off;
                const unsigned char *lp = sb + spr + lk_off;
                Real u[LNREAL];
#pragma unroll
                for (int v = 0; v < NVL; ++v) lds_vec(u + v * RPV, lp + (size_t)v * lk_str);
                if constexpr (LTAIL > 0) {
                    const Real *tp = reinterpret_cast<const Real *>(sb + spr + lkr) + (size_t)jl * LTAIL;
#pragma unroll
                    for (int e = 0; e < LTAIL; ++e) u[NVL * RPV + e] = tp[e];
                }
                auto release = [&]() {
                    __syncwarp();
                    if (lane == 0) mbar_arrive(empty0 + 8 * stage);
                };
                if constexpr (EARLY) {
                    Real psi[8 * D];
#pragma unroll
                    for (int v = 0; v < NVS; ++v) lds_vec(psi + v * RPV, sp + (size_t)v * sp_str);
                    release();
                    with_link<D, LK, Real>(u, [&](auto lk_c, const Real *ul) {
                        constexpr int K = decltype(lk_c)::value;
                        hop_component<MU, DIR, D, K, Real>(ul, psi + 0 * 2 * D, psi + P0 * 2 * D, (Real)1, sgn, acc[0], acc[P0]);
                        hop_component<MU, DIR, D, K, Real>(ul, psi + 1 * 2 * D, psi + P1 * 2 * D, (Real)(MU >= 2 ? -1 : 1), sgn, acc[1], acc[P1]);
                    });
                } else {
                    // large sites: one half-spinor component at a time, so that only 4 d_R spinor reals are live
                    with_link<D, LK, Real>(u, [&](auto lk_c, const Real *ul) {
                        constexpr int K = decltype(lk_c)::value;
                        Real pa[2 * D], pq[2 * D];
#pragma unroll
                        for (int v = 0; v < SPV; ++v) {
                            lds_vec(pa + v * RPV, sp + (size_t)(0 * SPV + v) * sp_str);
                            lds_vec(pq + v * RPV, sp + (size_t)(P0 * SPV + v) * sp_str);
                        }
                        hop_component<MU, DIR, D, K, Real>(ul, pa, pq, (Real)1, sgn, acc[0], acc[P0]);
#pragma unroll
                        for (int v = 0; v < SPV; ++v) {
                            lds_vec(pa + v * RPV, sp + (size_t)(1 * SPV + v) * sp_str);
                            lds_vec(pq + v * RPV, sp + (size_t)(P1 * SPV + v) * sp_str);
                        }
                        release();
                        hop_component<MU, DIR, D, K, Real>(ul, pa, pq, (Real)(MU >= 2 ? -1 : 1), sgn, acc[1], acc[P1]);
                    });
                }
                advance();
            };
            using I0 = std::integral_constant<int, 0>; using I1 = std::integral_constant<int, 1>;
            using I2 = std::integral_constant<int, 2>; using I3 = std::integral_constant<int, 3>;
            hop(I0{}, I0{}); hop(I0{}, I1{});
            hop(I1{}, I0{}); hop(I1{}, I1{});
            hop(I2{}, I0{}); hop(I2{}, I1{});
            hop(I3{}, I0{}); hop(I3{}, I1{});

            // epilogue (a6): as dphi_kernel
            Real o[8 * D];
            if constexpr (MASS) {
                const Real be[2] = { coef_beta<Real>(a, 0), coef_beta<Real>(a, 1) };
                Real self[8 * D];
                load_record<LD_STREAM, 8 * D>(self, (const char *)a.self, vh, s, 0);
                const Real al_[2] = { coef_alpha<Real>(a, 0), coef_alpha<Real>(a, 1) };
#pragma unroll
                for (int al = 0; al < 4; ++al)
#pragma unroll
                    for (int c = 0; c < 2 * D; ++c) o[al * 2 * D + c] = fma(al_[al >> 1], self[al * 2 * D + c], be[al >> 1] * acc[al][c]);
                if constexpr (RED) {
                    if (mine) {
#pragma unroll
                        for (int e = 0; e < 4 * D; ++e) {
                            const Real sr = self[2 * e], si = self[2 * e + 1], orr = o[2 * e], oi = o[2 * e + 1];
                            n2 = fma(orr, orr, fma(oi, oi, n2));
                            dre = fma(sr, orr, fma(si, oi, dre));
                            dim = fma(sr, oi, fma(-si, orr, dim));
                        }
                    }
                }
            } else {
#pragma unroll
                for (int al = 0; al < 4; ++al)
#pragma unroll
                    for (int c = 0; c < 2 * D; ++c) o[al * 2 * D + c] = (Real)-0.5 * acc[al][c];
            }
            if (mine) store_planes<ST_DEFAULT, 8 * D / RPV>((char *)a.out + s * 16, pb, o);
            }
        }
    }
    if constexpr (RED) {
        // the per-thread sums run over all tiles of this CTA; the producer warp contributes zeros
        double v[3] = { (double)n2, (double)dre, (double)dim };
        if (grid_reduce<3>(v, a.red_partial, a.red_ticket)) { a.red_result[0] = v[0]; a.red_result[1] = v[1]; a.red_result[2] = v[2]; }
    }
}

// host: tile geometry for this lattice, or false if the copies cannot be aligned (tail planes need 16-byte runs, the
// gauge field's per-direction stride must be a multiple of 16 bytes)
template <typename Real, int D, int LK>
static bool bulk_geometry(const DphiArgs &a, BulkArgs &g, size_t smem_max, int want_rows, int want_stages, int maxn = BulkGeom<Real, D, LK>::MAXN)
{
    using G = BulkGeom<Real, D, LK>;
    if (a.Zh > maxn) return false;
    if (G::TAILB != 0 && ((a.Zh * G::TAILB) % 16) != 0) return false;
    if ((((size_t)a.vh * G::TAILB) % 16) != 0) return false;
    int R = 0;
    for (int r = 1; r <= a.Y; ++r) {
        if (a.Y % r) continue;
        if (r * a.Zh > maxn) break;
        if (2 * (size_t)G::stage_bytes(r * a.Zh) + 256 > smem_max) break;
        if (want_rows > 0 && r > want_rows) break;
        R = r;
    }
    if (R == 0) return false;
    g.R = R;
    g.n = R * a.Zh;
    g.tiles_y = a.Y / R;
    g.ntiles = (long)a.T * a.X * g.tiles_y;
    g.stage_bytes = G::stage_bytes(g.n);
    int ns = (int)((smem_max - 256) / g.stage_bytes);
    if (ns > 8) ns = 8;
    if (want_stages >= 2 && want_stages < ns) ns = want_stages;
    g.nstage = ns;
    return ns >= 2;
}

struct BulkTuning { int rows, stages, ctas; }; // hr_ctx_set_tuning keys bulk_rows / bulk_stages / bulk_ctas; 0 = default

template <typename Real, int D, int LK, bool MASS, bool RED, int KS = 1>
static hr_status launch_bulk(const DphiArgs &a, cudaStream_t st, const BulkTuning &tn)
{
    using G = BulkGeom<Real, D, LK>;
    auto kern = dphi_bulk_kernel<Real, D, LK, MASS, RED, KS>;
    static bool attr_set[64] = {};
    static int sm_count[64] = {};
    static size_t dyn_max[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) { set_error("bulk kernel: device index %d", dev); return HR_EUNSUPPORTED; }
    if (!attr_set[dev]) {
        cudaFuncAttributes fa;
        cudaError_t e = cudaFuncGetAttributes(&fa, kern);
        if (e != cudaSuccess) { set_error("bulk kernel: cudaFuncGetAttributes: %s", cudaGetErrorString(e)); cudaGetLastError(); return HR_ECUDA; }
        dyn_max[dev] = kMaxDynSmem - ((fa.sharedSizeBytes + 1023) / 1024) * 1024;      // the fused reduction has static shared memory
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_max[dev]);
        if (e != cudaSuccess) { set_error("bulk kernel: cudaFuncSetAttribute: %s", cudaGetErrorString(e)); cudaGetLastError(); return HR_ECUDA; }
        cudaDeviceGetAttribute(&sm_count[dev], cudaDevAttrMultiProcessorCount, dev);
        attr_set[dev] = true;
    }
    const int ctas = tn.ctas > 0 ? tn.ctas : 1;
    BulkArgs g;
    // two threads per site: 7 consumer warps at most, so that a CTA of 256 threads keeps the whole register file
    if (!bulk_geometry<Real, D, LK>(a, g, dyn_max[dev] / ctas - 1024 * (ctas - 1), tn.rows, tn.stages, KS == 1 ? G::MAXN : 112)) {
        set_error("bulk kernel: no aligned tile for Zh=%d, Y=%d (d_R=%d)", a.Zh, a.Y, D);
        return HR_EUNSUPPORTED;
    }
    BulkMaps maps;
    constexpr size_t LB = (size_t)G::LNREAL * sizeof(Real);
    const int boxes[3] = { g.n, a.Zh, g.n - a.Zh };
    for (int k = 0; k < 3; ++k) {
        if (boxes[k] <= 0) { maps.sp[k] = maps.sp[0]; maps.lk[k] = maps.lk[0]; continue; }   // R = 1: never used
        hr_status r = encode_plane_map(&maps.sp[k], a.in, (size_t)a.vh, G::NVS, 1, 0, boxes[k]);
        if (r == HR_OK) r = encode_plane_map(&maps.lk[k], a.links, (size_t)a.vh, G::NVL, 8, LB * (size_t)a.vh, boxes[k]);
        if (r != HR_OK) return r;
    }
    const size_t smem = (size_t)g.nstage * g.stage_bytes + 2 * 8 * (size_t)g.nstage;
    long grid = (long)sm_count[dev] * ctas;
    if (grid > g.ntiles) grid = g.ntiles;
    const int block = 32 + ((KS * g.n + 31) / 32) * 32;
    kern<<<(unsigned)grid, block, smem, st>>>(a, g, maps);
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { set_error("dphi bulk kernel launch failed: %s", cudaGetErrorString(e)); return HR_ECUDA; }
    return HR_OK;
}

} // namespace hr
