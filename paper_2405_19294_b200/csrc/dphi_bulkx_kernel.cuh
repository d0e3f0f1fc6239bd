// dphi_bulkx_kernel.cuh -- Dphi_eo with the neighbour spinors staged in shared memory AND RE-USED ACROSS SITES: kernel
// variant 9 `bulkx` (north_star: "TMA or shared-memory staging of neighbour spinors along the fastest lattice direction
// so they are reused across sites").
//
// Why: under the 1 kW power cap a B200 runs this operator at ~1.4 GHz, and there the site kernel and the per-hop staged
// kernel (dphi_bulk_kernel.cuh) are bound by the L2 -> SM crossbar, not by HBM: they pull 8 links + 7-8 neighbour spinors
// per site through it (2.2-2.7 KB per site for SU(3) fundamental in fp64 against 1.5 KB of compulsory DRAM traffic;
// profiles/r2_staging.md).  Six of a site's eight neighbours lie in the same time-slice; a CTA that walks along x keeps
// them in shared memory:
//
//  * a TILE is R z-rows (n = R * Zh sites) of one (t, x); a CTA processes a STRIP of Lx tiles x0 .. x0+Lx-1 at fixed
//    (t, y0).  The input spinors of the time-slice live in BLOCKS: block(x) = rows y0-1 .. y0+R of column x (the R rows
//    of the tile plus one halo row on either side: three TMA boxes).  Tile x reads block(x-1) for the -x hop, block(x+1)
//    for the +x hop and block(x) for the +-y and +-z hops; moving on to x+1 only block(x+2) is new.  Three block slots
//    form a ring of their own: the slot of block(x-1) is released right after the -x hop of tile x and refilled with
//    block(x+2) while the +-y, +-z hops of this tile and the +-t hops of the next one run.
//  * the +-t neighbours (no re-use inside a time-slice) and the eight links of a site go through per-hop rings exactly
//    as in dphi_bulk_kernel.cuh.
//  * spinor bytes through the crossbar per site: (1 + 2/R)(1 + 2/Lx) + 2 spinors instead of 8.
//
// Producer = one elected lane of warp 0; consumers = one thread per site (KS = 1) or two (KS = 2, one per half-spinor
// component; the default in fp64 where a tile is only 64 sites).  Compiled for d_R <= 4 (the crossbar-bound kernels).
#pragma once
#include "dphi_bulk_kernel.cuh"

namespace hr {

struct BulkxArgs {
    int R, n;             // rows / sites per tile
    int Lx;               // tiles per strip (divides Xb)
    int tiles_y;          // Y / R
    int strips_x;         // Xb / Lx
    long nstrips;         // (X / Lx) * T * tiles_y
    int nt, nl;           // depth of the +-t spinor ring and of the link ring
    unsigned block_bytes, tslot_bytes, lslot_bytes;
};

enum { BULKX_NB = 3 };    // block slots: x-1, x, x+1; the slot of x-1 is released right after the -x hop and refilled with x+2

template <typename Real, int D, int LK> struct BulkxGeom {
    using G = BulkGeom<Real, D, LK>;
    __host__ __device__ static constexpr unsigned halo_bytes(int zh) { return bulk_r128((unsigned)(G::NVS * zh * 16)); }
    __host__ __device__ static constexpr unsigned core_bytes(int n) { return bulk_r128((unsigned)(G::NVS * n * 16)); }
    __host__ __device__ static constexpr unsigned block_bytes(int n, int zh) { return 2 * halo_bytes(zh) + core_bytes(n); }
    __host__ __device__ static constexpr unsigned tslot_bytes(int n) { return core_bytes(n); }
    __host__ __device__ static constexpr unsigned lslot_bytes(int n)
    {
        return bulk_r128(G::lk_region(n) + (((unsigned)(n * G::TAILB) + 15u) & ~15u));
    }
};

template <typename Real, int D, int LK, bool MASS, bool RED, int KS>
__global__ void __launch_bounds__((KS == 1 ? 32 + BulkGeom<Real, D, LK>::MAXN : 256), 1)
dphi_bulkx_kernel(const DphiArgs a, const BulkxArgs g, const __grid_constant__ BulkMaps maps)
{
    using G = BulkGeom<Real, D, LK>;
    using GX = BulkxGeom<Real, D, LK>;
    constexpr int RPV = G::RPV, LNREAL = G::LNREAL, NVS = G::NVS, NVL = G::NVL, LTAIL = G::LTAIL;
    constexpr int SPV = 2 * D / RPV;
    static_assert(KS == 1 || (2 * D) % RPV == 0, "two threads per site need vector-aligned spin components");
    static_assert(D <= 4, "bulkx: small sites only (whole stage read, then released)");
    extern __shared__ __align__(128) unsigned char smem[];
    if (a.skip != nullptr && *a.skip != 0) return;

    const int n = g.n, Zh = a.Zh, R = g.R, nt = g.nt, nl = g.nl;
    const unsigned halo_b = GX::halo_bytes(Zh), core_b = GX::core_bytes(n);
    unsigned char *blk0 = smem;
    unsigned char *tsl0 = blk0 + (size_t)BULKX_NB * g.block_bytes;
    unsigned char *lsl0 = tsl0 + (size_t)nt * g.tslot_bytes;
    uint64_t *bars = reinterpret_cast<uint64_t *>(lsl0 + (size_t)nl * g.lslot_bytes);
    // barriers: [full_b NB][empty_b NB][full_t nt][empty_t nt][full_l nl][empty_l nl]
    const uint32_t fullb = smem_addr(bars), emptyb = fullb + 8 * BULKX_NB;
    const uint32_t fullt = emptyb + 8 * BULKX_NB, emptyt = fullt + 8 * nt;
    const uint32_t fulll = emptyt + 8 * nt, emptyl = fulll + 8 * nl;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ncw = (int)(blockDim.x >> 5) - 1;
    if (threadIdx.x == 0) {
        for (int k = 0; k < BULKX_NB; ++k) { mbar_init(fullb + 8 * k, 1); mbar_init(emptyb + 8 * k, (uint32_t)ncw); }
        for (int k = 0; k < nt; ++k) { mbar_init(fullt + 8 * k, 1); mbar_init(emptyt + 8 * k, (uint32_t)ncw); }
        for (int k = 0; k < nl; ++k) { mbar_init(fulll + 8 * k, 1); mbar_init(emptyl + 8 * k, (uint32_t)ncw); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    const size_t vh = (size_t)a.vh;
    const size_t pb = vh * 16;
    constexpr size_t LB = (size_t)LNREAL * sizeof(Real);
    const long rowst = Zh, st_x = (long)a.Y * Zh, st_t = (long)a.X * a.Y * Zh;

    // strip -> (t, x0, y0); strips are ordered [x / Xb][t][(x % Xb) / Lx][y0 / R]: the x-blocked order of dphi_kernel
    auto decode = [&](long strip, int &t, int &x0, int &y0) {
        unsigned r = (unsigned)strip;
        const int yb = (int)(r % (unsigned)g.tiles_y); r /= (unsigned)g.tiles_y;
        const int sx = (int)(r % (unsigned)g.strips_x); r /= (unsigned)g.strips_x;
        t = (int)(r % (unsigned)a.T);
        x0 = (int)(r / (unsigned)a.T) * a.Xb + sx * g.Lx;
        y0 = yb * R;
    };

    unsigned qb = 0;                      // block sequence number: slot = q % NB, phase = (q / NB) & 1
    auto bslot = [](unsigned q) { return q % (unsigned)BULKX_NB; };
    auto bphase = [](unsigned q) { return (q / (unsigned)BULKX_NB) & 1u; };
    int ts = 0, ls = 0;                   // slots of the +-t ring and of the link ring
    uint32_t tph = 0, lph = 0;
    auto adv_t = [&]() { if (++ts == nt) { ts = 0; tph ^= 1u; } };
    auto adv_l = [&]() { if (++ls == nl) { ls = 0; lph ^= 1u; } };

    [[maybe_unused]] Real n2 = 0, dre = 0, dim = 0;

    if (warp == 0) {
        // =============================== producer ===============================
        if (lane == 0) {
            const uint32_t blk_tx = (uint32_t)(n + 2 * Zh) * NVS * 16u, t_tx = (uint32_t)n * NVS * 16u;
            const uint32_t l_tx = (uint32_t)n * (uint32_t)(NVL * 16 + G::TAILB);
            const char *tail0 = (const char *)a.links + (size_t)NVL * 16 * vh;
            for (long strip = blockIdx.x; strip < g.nstrips; strip += gridDim.x) {
                int t, x0, y0;
                decode(strip, t, x0, y0);
                const int ylo = y0 == 0 ? a.Y - 1 : y0 - 1, yhi = y0 + R == a.Y ? 0 : y0 + R;
                auto issue_block = [&](int xx) {
                    const int xw = xx < 0 ? xx + a.X : (xx >= a.X ? xx - a.X : xx);
                    const long col = ((long)t * a.X + xw) * a.Y;
                    const unsigned slot = bslot(qb);
                    mbar_wait(emptyb + 8 * slot, bphase(qb) ^ 1u);
                    const uint32_t fb = fullb + 8 * slot;
                    mbar_arrive_expect_tx(fb, blk_tx);
                    const uint32_t dst = smem_addr(blk0 + (size_t)slot * g.block_bytes);
                    tma_2d(dst, &maps.sp[1], (int)(2 * (col + ylo) * Zh), fb);
                    tma_2d(dst + halo_b, &maps.sp[0], (int)(2 * (col + y0) * Zh), fb);
                    tma_2d(dst + halo_b + core_b, &maps.sp[1], (int)(2 * (col + yhi) * Zh), fb);
                    ++qb;
                };
                issue_block(x0 - 1);
                issue_block(x0);
                for (int jx = 0; jx < g.Lx; ++jx) {
                    const int x = x0 + jx;
                    const long s0 = (((long)t * a.X + x) * a.Y + y0) * Zh;
#pragma unroll 1
                    for (int h = 0; h < 8; ++h) {
                        const int mu = h >> 1, dir = h & 1;
                        if (h == 2) issue_block(x + 1);
                        long src0 = s0, src1 = 0;
                        int cnt0 = n, cnt1 = 0;
                        if (mu == 0) {
                            const int tn = dir == 0 ? (t == a.T - 1 ? 0 : t + 1) : (t == 0 ? a.T - 1 : t - 1);
                            src0 = s0 + (long)(tn - t) * st_t;
                            mbar_wait(emptyt + 8 * ts, tph ^ 1u);
                            mbar_arrive_expect_tx(fullt + 8 * ts, t_tx);
                            tma_2d(smem_addr(tsl0 + (size_t)ts * g.tslot_bytes), &maps.sp[0], (int)(2 * src0), fullt + 8 * ts);
                            adv_t();
                        } else if (mu == 1) {
                            const int xn = dir == 0 ? (x == a.X - 1 ? 0 : x + 1) : (x == 0 ? a.X - 1 : x - 1);
                            src0 = s0 + (long)(xn - x) * st_x;
                        } else if (mu == 2 && dir == 1) {
                            if (y0 > 0) src0 = s0 - rowst;
                            else if (R == 1) src0 = s0 + (long)(a.Y - 1) * rowst;
                            else { src0 = s0 + (long)(a.Y - 1) * rowst; cnt0 = Zh; src1 = s0; cnt1 = n - Zh; }
                        }
                        // link box(es): the forward hop reads the tile's own links, the backward hop the neighbours'
                        const int field = (dir == 0 ? a.parity : 1 - a.parity) * 4 + mu;
                        mbar_wait(emptyl + 8 * ls, lph ^ 1u);
                        const uint32_t fb = fulll + 8 * ls;
                        mbar_arrive_expect_tx(fb, l_tx);
                        const uint32_t lbase = smem_addr(lsl0 + (size_t)ls * g.lslot_bytes);
                        const bool split = dir == 1 && cnt1 != 0;
                        if (!split) tma_3d(lbase, &maps.lk[0], (int)(2 * (dir == 0 ? s0 : src0)), field, fb);
                        else {
                            tma_3d(lbase, &maps.lk[1], (int)(2 * src0), field, fb);
                            tma_3d(lbase + bulk_r128((unsigned)(NVL * Zh * 16)), &maps.lk[2], (int)(2 * src1), field, fb);
                        }
                        if constexpr (LTAIL > 0) {
                            const char *tf = tail0 + (size_t)field * LB * vh;
                            const uint32_t tb = lbase + G::lk_region(n);
                            if (!split) bulk_g2s(tb, tf + (size_t)(dir == 0 ? s0 : src0) * G::TAILB, (uint32_t)(n * G::TAILB), fb);
                            else {
                                bulk_g2s(tb, tf + (size_t)src0 * G::TAILB, (uint32_t)(cnt0 * G::TAILB), fb);
                                bulk_g2s(tb + (uint32_t)(cnt0 * G::TAILB), tf + (size_t)src1 * G::TAILB, (uint32_t)(cnt1 * G::TAILB), fb);
                            }
                        }
                        adv_l();
                    }
                }
            }
        }
    } else {
        // =============================== consumers ===============================
        const int ic = ((int)threadIdx.x - 32) / KS;
        [[maybe_unused]] const int kk = ((int)threadIdx.x - 32) % KS;   // KS = 2: my half-spinor component
        const bool mine = ic < n;
        const int i = mine ? ic : n - 1;                      // idle lanes shadow the last site (no stores)
        const int row = i / Zh, zh = i - row * Zh;
        const unsigned cC = (unsigned)(n - Zh);

        for (long strip = blockIdx.x; strip < g.nstrips; strip += gridDim.x) {
            int t, x0, y0;
            decode(strip, t, x0, y0);
            const int y = y0 + row;
            // the first two blocks of the strip
            mbar_wait(fullb + 8 * bslot(qb), bphase(qb));
            mbar_wait(fullb + 8 * bslot(qb + 1), bphase(qb + 1));
            for (int jx = 0; jx < g.Lx; ++jx, ++qb) {
                const int x = x0 + jx;
                const int b = (t + x + y + a.parity) & 1;
                const size_t s = (size_t)((((long)t * a.X + x) * a.Y + y0) * Zh + i);
                const unsigned char *blk_m = blk0 + (size_t)bslot(qb) * g.block_bytes;          // column x-1
                const unsigned char *blk_c = blk0 + (size_t)bslot(qb + 1) * g.block_bytes;      // column x
                const unsigned char *blk_p = blk0 + (size_t)bslot(qb + 2) * g.block_bytes;      // column x+1

                // accumulators: KS = 1: acc[0..3] = out_0..3.  KS = 2: acc[0] -> out_k, acc[1] -> out_{k+2} (mu = 0,3),
                // acc[2] -> out_{3-k} (mu = 1,2; handed to the partner lane at the end)
                constexpr int NACC = KS == 1 ? 4 : 3;
                Real acc[NACC][2 * D];
#pragma unroll
                for (int al = 0; al < NACC; ++al)
#pragma unroll
                    for (int c = 0; c < 2 * D; ++c) acc[al][c] = 0;

                auto hop = [&](auto mu_c, auto dir_c) {
                    constexpr int MU = decltype(mu_c)::value;
                    constexpr int DIR = decltype(dir_c)::value;
                    int j = i, sign = 1;
                    const unsigned char *sp;                      // my vector of plane 0 of the neighbour spinor
                    unsigned sp_str = (unsigned)n * 16u;          // plane stride
                    unsigned lk_off, lk_str = (unsigned)n * 16u;
                    if constexpr (MU == 0) {
                        sign = (DIR == 0 ? t == a.T - 1 : t == 0) ? a.bc[0] : 1;
                        mbar_wait(fullt + 8 * ts, tph);
                        sp = tsl0 + (size_t)ts * g.tslot_bytes + (size_t)i * 16;
                    } else if constexpr (MU == 1) {
                        sign = (DIR == 0 ? x == a.X - 1 : x == 0) ? a.bc[1] : 1;
                        if constexpr (DIR == 0) mbar_wait(fullb + 8 * bslot(qb + 2), bphase(qb + 2));   // the new block
                        sp = (DIR == 0 ? blk_p : blk_m) + halo_b + (size_t)i * 16;
                    } else if constexpr (MU == 2) {
                        sign = (DIR == 0 ? y == a.Y - 1 : y == 0) ? a.bc[2] : 1;
                        if constexpr (DIR == 0) {
                            if (row < R - 1) sp = blk_c + halo_b + (size_t)(i + Zh) * 16;
                            else { sp = blk_c + halo_b + core_b + (size_t)zh * 16; sp_str = (unsigned)Zh * 16u; }
                        } else {
                            if (row > 0) sp = blk_c + halo_b + (size_t)(i - Zh) * 16;
                            else { sp = blk_c + (size_t)zh * 16; sp_str = (unsigned)Zh * 16u; }
                        }
                    } else {
                        if constexpr (DIR == 0) {
                            const bool w = zh == Zh - 1;
                            j = b ? (w ? i - (Zh - 1) : i + 1) : i;
                            sign = (b && w) ? a.bc[3] : 1;
                        } else {
                            const bool w = zh == 0;
                            j = b ? i : (w ? i + (Zh - 1) : i - 1);
                            sign = (!b && w) ? a.bc[3] : 1;
                        }
                        sp = blk_c + halo_b + (size_t)j * 16;
                    }
                    lk_off = (unsigned)(DIR == 0 ? i : j) * 16u;
                    if constexpr (MU == 2 && DIR == 1) {
                        if (R > 1 && y0 == 0) {                   // link boxes: [row y = Y-1][tile less its first row]
                            if (row == 0) lk_str = (unsigned)Zh * 16u;
                            else { lk_off = bulk_r128((unsigned)(NVL * Zh) * 16u) + (unsigned)(i - Zh) * 16u; lk_str = cC * 16u; }
                        }
                    }
                    [[maybe_unused]] const int jl = DIR == 0 ? i : j;
                    const Real sgn = (Real)sign;

                    mbar_wait(fulll + 8 * ls, lph);
                    const unsigned char *lb = lsl0 + (size_t)ls * g.lslot_bytes;
                    const unsigned char *lp = lb + lk_off;
                    Real u[LNREAL];
#pragma unroll
                    for (int v = 0; v < NVL; ++v) lds_vec(u + v * RPV, lp + (size_t)v * lk_str);
                    if constexpr (LTAIL > 0) {
                        const Real *tp = reinterpret_cast<const Real *>(lb + G::lk_region(n)) + (size_t)jl * LTAIL;
#pragma unroll
                        for (int e = 0; e < LTAIL; ++e) u[NVL * RPV + e] = tp[e];
                    }
                    auto release = [&]() {
                        __syncwarp();
                        if (lane == 0) {
                            mbar_arrive(emptyl + 8 * ls);
                            if constexpr (MU == 0) mbar_arrive(emptyt + 8 * ts);
                            if constexpr (MU == 1 && DIR == 1) mbar_arrive(emptyb + 8 * bslot(qb));   // column x-1: last use
                        }
                    };
                    if constexpr (KS == 1) {
                        constexpr int P0 = (MU == 0 || MU == 3) ? 2 : 3;
                        constexpr int P1 = 5 - P0;
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
                        constexpr bool STRAIGHT = (MU == 0 || MU == 3);
                        const int pk = STRAIGHT ? kk + 2 : 3 - kk;
                        Real pa[2 * D], pq[2 * D];
#pragma unroll
                        for (int v = 0; v < SPV; ++v) {
                            lds_vec(pa + v * RPV, sp + (size_t)(kk * SPV + v) * sp_str);
                            lds_vec(pq + v * RPV, sp + (size_t)(pk * SPV + v) * sp_str);
                        }
                        release();
                        const Real sk = (MU >= 2 && kk == 1) ? (Real)-1 : (Real)1;
                        with_link<D, LK, Real>(u, [&](auto lk_c, const Real *ul) {
                            hop_component<MU, DIR, D, decltype(lk_c)::value, Real>(ul, pa, pq, sk, sgn, acc[0], acc[STRAIGHT ? 1 : 2]);
                        });
                    }
                    if constexpr (MU == 0) adv_t();
                    adv_l();
                };
                using I0 = std::integral_constant<int, 0>; using I1 = std::integral_constant<int, 1>;
                using I2 = std::integral_constant<int, 2>; using I3 = std::integral_constant<int, 3>;
                hop(I0{}, I0{}); hop(I0{}, I1{});
                hop(I1{}, I0{}); hop(I1{}, I1{});
                hop(I2{}, I0{}); hop(I2{}, I1{});
                hop(I3{}, I0{}); hop(I3{}, I1{});

                // at the end of a strip the other two blocks are done with as well
                if (jx == g.Lx - 1) {
                    __syncwarp();
                    if (lane == 0) { mbar_arrive(emptyb + 8 * bslot(qb + 1)); mbar_arrive(emptyb + 8 * bslot(qb + 2)); }
                }

                // epilogue (a6): as dphi_kernel
                if constexpr (KS == 1) {
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
                } else {
                    Real *accK = acc[0], *accP = acc[1], *accQ = acc[2];
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
                }
            }
            qb += 2;                      // a strip of Lx tiles used Lx + 2 blocks
        }
    }
    if constexpr (RED) {
        double v[3] = { (double)n2, (double)dre, (double)dim };
        if (grid_reduce<3>(v, a.red_partial, a.red_ticket)) { a.red_result[0] = v[0]; a.red_result[1] = v[1]; a.red_result[2] = v[2]; }
    }
}

// host: strip / tile geometry and the split of shared memory between the block slots and the two rings
template <typename Real, int D, int LK>
static bool bulkx_geometry(const DphiArgs &a, BulkxArgs &g, size_t smem_max, int want_rows, int want_strip, int maxn, long grid)
{
    using G = BulkGeom<Real, D, LK>;
    using GX = BulkxGeom<Real, D, LK>;
    if (a.Zh > maxn) return false;
    if (G::TAILB != 0 && ((a.Zh * G::TAILB) % 16) != 0) return false;
    if ((((size_t)a.vh * G::TAILB) % 16) != 0) return false;
    int R = 0;
    for (int r = 1; r <= a.Y; ++r) {
        if (a.Y % r) continue;
        if (r * a.Zh > maxn) break;
        // the block slots + at least 2 +-t slots and 3 link slots
        const size_t need = (size_t)BULKX_NB * GX::block_bytes(r * a.Zh, a.Zh) + 2 * (size_t)GX::tslot_bytes(r * a.Zh) +
                            3 * (size_t)GX::lslot_bytes(r * a.Zh) + 512;
        if (need > smem_max) break;
        if (want_rows > 0 && r > want_rows) break;
        R = r;
    }
    if (R == 0) return false;
    g.R = R;
    g.n = R * a.Zh;
    g.tiles_y = a.Y / R;
    // strip length: the longest divisor of Xb (<= 16) that still leaves every CTA six strips or more
    int Lx = 1;
    for (int l = 1; l <= a.Xb && l <= 16; ++l) {
        if (a.Xb % l) continue;
        if (want_strip > 0) { if (l <= want_strip) Lx = l; continue; }
        const long ns = (long)(a.X / l) * a.T * g.tiles_y;
        if (l <= 4 || ns >= 6 * grid) Lx = l;
    }
    g.Lx = Lx;
    g.strips_x = a.Xb / Lx;
    g.nstrips = (long)(a.X / Lx) * a.T * g.tiles_y;
    g.block_bytes = GX::block_bytes(g.n, a.Zh);
    g.tslot_bytes = GX::tslot_bytes(g.n);
    g.lslot_bytes = GX::lslot_bytes(g.n);
    // the rest of shared memory goes to the two rings (a tile uses 2 +-t slots and 8 link slots): the deepest pair that fits
    const size_t rest = smem_max - 512 - (size_t)BULKX_NB * g.block_bytes;
    static const int kRings[][2] = { { 2, 3 }, { 2, 4 }, { 2, 5 }, { 2, 6 }, { 3, 6 }, { 3, 7 }, { 3, 8 }, { 3, 9 }, { 4, 9 }, { 4, 10 }, { 4, 11 }, { 4, 12 } };
    int nt = 2, nl = 3;
    for (const auto &rg : kRings)
        if ((size_t)rg[0] * g.tslot_bytes + (size_t)rg[1] * g.lslot_bytes <= rest) { nt = rg[0]; nl = rg[1]; }
    g.nt = nt;
    g.nl = nl;
    return true;
}

template <typename Real, int D, int LK, bool MASS, bool RED, int KS>
static hr_status launch_bulkx(const DphiArgs &a, cudaStream_t st, const BulkTuning &tn, int want_strip)
{
    using G = BulkGeom<Real, D, LK>;
    auto kern = dphi_bulkx_kernel<Real, D, LK, MASS, RED, KS>;
    static bool attr_set[64] = {};
    static int sm_count[64] = {};
    static size_t dyn_max[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) { set_error("bulkx kernel: device index %d", dev); return HR_EUNSUPPORTED; }
    if (!attr_set[dev]) {
        cudaFuncAttributes fa;
        cudaError_t e = cudaFuncGetAttributes(&fa, kern);
        if (e != cudaSuccess) { set_error("bulkx kernel: cudaFuncGetAttributes: %s", cudaGetErrorString(e)); cudaGetLastError(); return HR_ECUDA; }
        dyn_max[dev] = kMaxDynSmem - ((fa.sharedSizeBytes + 1023) / 1024) * 1024;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_max[dev]);
        if (e != cudaSuccess) { set_error("bulkx kernel: cudaFuncSetAttribute: %s", cudaGetErrorString(e)); cudaGetLastError(); return HR_ECUDA; }
        cudaDeviceGetAttribute(&sm_count[dev], cudaDevAttrMultiProcessorCount, dev);
        attr_set[dev] = true;
    }
    BulkxArgs g;
    long grid = sm_count[dev];
    if (!bulkx_geometry<Real, D, LK>(a, g, dyn_max[dev], tn.rows, want_strip, KS == 1 ? G::MAXN : 112, grid)) {
        set_error("bulkx kernel: no tile fits shared memory / alignment for Zh=%d, Y=%d (d_R=%d)", a.Zh, a.Y, D);
        return HR_EUNSUPPORTED;
    }
    BulkMaps maps;
    constexpr size_t LB = (size_t)G::LNREAL * sizeof(Real);
    const int boxes[3] = { g.n, a.Zh, g.n - a.Zh };
    for (int k = 0; k < 3; ++k) {
        if (boxes[k] <= 0) { maps.sp[k] = maps.sp[0]; maps.lk[k] = maps.lk[0]; continue; }
        hr_status r = encode_plane_map(&maps.sp[k], a.in, (size_t)a.vh, G::NVS, 1, 0, boxes[k]);
        if (r == HR_OK) r = encode_plane_map(&maps.lk[k], a.links, (size_t)a.vh, G::NVL, 8, LB * (size_t)a.vh, boxes[k]);
        if (r != HR_OK) return r;
    }
    const size_t smem = (size_t)BULKX_NB * g.block_bytes + (size_t)g.nt * g.tslot_bytes + (size_t)g.nl * g.lslot_bytes +
                        8 * 2 * (size_t)(BULKX_NB + g.nt + g.nl);
    if (grid > g.nstrips) grid = g.nstrips;
    const int block = 32 + ((KS * g.n + 31) / 32) * 32;
    kern<<<(unsigned)grid, block, smem, st>>>(a, g, maps);
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { set_error("dphi bulkx kernel launch failed: %s", cudaGetErrorString(e)); return HR_ECUDA; }
    return HR_OK;
}

} // namespace hr
