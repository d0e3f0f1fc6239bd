// dphi_cp_kernel.cuh -- the COLOUR-PARALLEL Dphi kernel (kernel variant 6, "colour"): one thread per (site, colour row).
//
// The paper's answer to large fermion representations (section 3.1.2): when d_R grows, a thread that owns
// a whole site holds 8 d_R accumulators, a 8 d_R spinor and a d_R x d_R link and spills ("the unimproved kernel blows
// up"); its LARGE_N kernel parallelises over the fermion dimension instead.  The sm_100a form of that idea:
//
//   * a CTA owns SITES = 32 consecutive half-indices; warp a of the CTA owns colour row a of all of them, so every
//     global access of a warp is one record element of 32 consecutive sites (coalesced in the plane layout of
//     hr_internal.h) and the d_R warps of a CTA read 32 whole records between them;
//   * per hop a thread loads only the four spin components of ITS colour of the neighbour spinor, projects them to
//     its two half-spinor entries h_{k,a} (k = 0,1) and puts them into shared memory; after a barrier it reads all h_{k,b}
//     back (conflict-free: consecutive lanes = consecutive sites) and multiplies with row a of U (forward hop) or
//     column a of U, conjugated (backward hop: row a of U^dagger);
//   * hops go in two batches of four (mu = 0,1 and mu = 2,3): 8 d_R half-spinor entries per site in shared memory
//     (d_R = 10, fp64: 40 KB per CTA), three barriers per launch;
//   * a thread carries 4 complex accumulators and O(d_R) link elements in flight, whatever d_R is: no spilling, the
//     occupancy no longer falls with d_R^2.
//
// Link kinds: the represented complex (LK_COMPLEX) or real (LK_REAL) field.  Epilogue, fused reduction and the skip flag
// are those of dphi_kernel (DphiArgs); the fused site matrix is not available here.
#pragma once
#include "dphi_kernel.cuh"

namespace hr {

// complex element e (in complex units) of site s of a record field of NREAL reals
template <int HINT, int NREAL>
__device__ __forceinline__ void load_cplx(double &re, double &im, const char *base, size_t vh, size_t s, int e, uint64_t pol)
{
    static_assert(NREAL % 2 == 0, "complex record");
    ld16<HINT>(re, im, base + ((size_t)e * vh + s) * 16, pol);
}
template <int HINT, int NREAL>
__device__ __forceinline__ void load_cplx(float &re, float &im, const char *base, size_t vh, size_t s, int e, uint64_t pol)
{
    static_assert(NREAL % 2 == 0, "complex record");
    constexpr int NV = NREAL / 4;
    if (NREAL % 4 == 0 || (e >> 1) < NV) ld8<HINT>(re, im, base + ((size_t)(e >> 1) * vh + s) * 16 + (size_t)(e & 1) * 8, pol);
    else ld8<HINT>(re, im, base + (size_t)NV * 16 * vh + s * 8, pol);                       // 8-byte tail plane
}
// real element e of site s of a record field of NREAL reals
template <int HINT, int NREAL>
__device__ __forceinline__ void load_real(double &r, const char *base, size_t vh, size_t s, int e, uint64_t pol)
{
    constexpr int NV = NREAL / 2;
    if (NREAL % 2 == 0 || (e >> 1) < NV) ld8<HINT>(r, base + ((size_t)(e >> 1) * vh + s) * 16 + (size_t)(e & 1) * 8, pol);
    else ld8<HINT>(r, base + (size_t)NV * 16 * vh + s * 8, pol);
}
template <int HINT, int NREAL>
__device__ __forceinline__ void load_real(float &r, const char *base, size_t vh, size_t s, int e, uint64_t pol)
{
    constexpr int NV = NREAL / 4, TAIL = NREAL - 4 * NV;
    if (TAIL == 0 || (e >> 2) < NV) ld4<HINT>(r, base + ((size_t)(e >> 2) * vh + s) * 16 + (size_t)(e & 3) * 4, pol);
    else ld4<HINT>(r, base + (size_t)NV * 16 * vh + s * (size_t)(TAIL * 4) + (size_t)(e - 4 * NV) * 4, pol);
}

// CNT consecutive elements (C reals each) of site s starting at element e0.  ALIGNED (the caller knows statically that
// the run starts and ends on 16-byte vectors): whole-vector loads; otherwise element by element.
template <int HINT, int NREAL, int C, int CNT, bool ALIGNED, typename Real>
__device__ __forceinline__ void load_elems(Real *dst, const char *base, size_t vh, size_t s, int e0)
{
    constexpr int RPV = 16 / (int)sizeof(Real);
    if constexpr (ALIGNED) {
        static_assert((CNT * C) % RPV == 0, "aligned run: whole vectors");
        load_planes<HINT, CNT * C / RPV>(dst, base + ((size_t)(e0 * C / RPV) * vh + s) * 16, vh * 16, 0);
    } else {
#pragma unroll
        for (int i = 0; i < CNT; ++i) {
            if constexpr (C == 2) load_cplx<HINT, NREAL>(dst[2 * i], dst[2 * i + 1], base, vh, s, e0 + i, 0);
            else load_real<HINT, NREAL>(dst[i], base, vh, s, e0 + i, 0);
        }
    }
}

template <typename Real> struct alignas(2 * sizeof(Real)) CpPair { Real re, im; };

template <typename Real, int D, bool RL> struct CpGeom {
    static constexpr int RPV = 16 / (int)sizeof(Real);
    static constexpr int C = RL ? 1 : 2;             // reals per link element
    static constexpr int EPV = RPV / C;              // link elements per 16-byte vector
    // colour rows per thread: 2 when that turns the spinor entries (fp32) and the column entries of a backward hop
    // (fp32 complex, fp64 real) into whole 16-byte vectors -- needs an even d_R; 1 otherwise.
    // PAD: real links of an odd d_R > 8 (SU(4) adjoint, 15 x 15) are stored with rows of LD = d_R + 1 reals (LinkGeom::LD).
    // With RPT = 4 (fp32) / 2 (fp64) rows per thread and r0 a multiple of RPT, both a thread's rows of U (forward hop) and
    // its RPT columns of every row of U (backward hop: rows of U^T) are whole 16-byte vectors at compile-time plane offsets
    // from one per-thread base.  The last row group is ragged (rows 12, 13, 14 and a dummy): the dummy row loads nothing,
    // holds zeros in the half-spinor exchange and stores nothing.
    // Before (round 1 / early round 2: unpadded rows, RPT = 1): every link element was a 4- / 8-byte load at a run-time
    // plane and word (12 integer instructions per load) and all 15 threads of a site re-read the 30 half-spinor entries of
    // a hop from shared memory (7.2 KB per site and hop in fp64 against 1.8 KB of link): L1 pipe 90 % busy, 0.74 (fp64) /
    // 0.50 (fp32; 0.55 with the links staged through shared memory by cp.async) of the copy peak.  Now, SU(4) adjoint
    // 16^3 x 48 on the UNPADDED 8L + 2S bytes: fp64 0.333 -> 0.281 ms (0.87), fp32 0.223 -> 0.150 ms (0.82); the padded
    // bytes cap that figure at 225 / 240 = 0.94.  Sweep (profiles/r2_large_n.md): fp64 RPT 2 / chunk 16 / 16 sites per CTA;
    // fp32 RPT 4 / chunk 8 / 32 sites; 128 registers (100 and 84 spill: 0.75 / 0.61; RPT = 4 in fp64 needs 168: 0.85).
#ifndef HR_CP_RPT_PAD64
#define HR_CP_RPT_PAD64 2
#endif
#ifndef HR_CP_RPT_PAD32
#define HR_CP_RPT_PAD32 4
#endif
#ifndef HR_CP_RPT
// two rows per thread for complex fp64 links too (a complex entry is already a whole vector; what is gained is half the
// shared-memory reads of the half-spinor exchange and two link rows in flight per thread): measured, SU(3) sextet 24^3 x 48
// 0.301 -> 0.290 ms (0.90 -> 0.94), SU(4) sextet d_R = 10 0.260 -> 0.264 ms -- so at d_R = 6 only
#ifndef HR_CP_RPT2_F64C
#define HR_CP_RPT2_F64C (D == 6)
#endif
#define HR_CP_RPT (PAD ? (sizeof(Real) == 8 ? HR_CP_RPT_PAD64 : HR_CP_RPT_PAD32) : (D % 2 == 0 && (sizeof(Real) == 4 || RL || HR_CP_RPT2_F64C)) ? 2 : 1)
#endif
    static constexpr int LD = LinkGeom<RL ? LK_REAL : LK_COMPLEX, D>::LD;
    static constexpr bool PAD = LD != D;
    static constexpr int RPT = HR_CP_RPT;
    static constexpr int NG = (D + RPT - 1) / RPT;   // row groups = threads per site
    static constexpr int DP = NG * RPT;              // colours in the half-spinor exchange (D, or D + dummies when PAD)
    static_assert(D % RPT == 0 || PAD, "rows per thread must divide d_R");
    static_assert(!PAD || (RPT % RPV == 0 && LD % RPV == 0), "padded rows: a thread's rows / columns must be whole vectors");
    // sites per CTA: a warp covers 32 sites of one row group, or (more than 12 groups, where 32 x groups threads would
    // leave one CTA per SM alone with its barriers; fp64 PAD: measured) 16 sites of two groups; THREADS is padded to whole
    // warps, the padding threads shadow the last group and store nothing
#ifndef HR_CP_SITES
#define HR_CP_SITES ((NG > 12 || (PAD && sizeof(Real) == 8)) ? 16 : 32)
#endif
    static constexpr int SITES = HR_CP_SITES;
    static constexpr int THREADS = (SITES * NG + 31) / 32 * 32;
    static constexpr int HB = 4;                     // hops per batch
    static constexpr int LNREAL_ = RL ? D * LD : 2 * D * D;
    __host__ __device__ static constexpr size_t hs_bytes() { return (size_t)HB * 2 * DP * SITES * sizeof(CpPair<Real>); }
    static constexpr size_t smem_bytes() { return hs_bytes(); }
    // registers: a thread's state does not grow with d_R, so the cap is chosen for occupancy (several CTAs per SM hide
    // the three barriers): HR_CP_REGS registers per thread per row
    // (measured on B200, bench_large_n: SU(4) sym d_R = 10 fp64 0.260 ms at 84, 0.275 at 160, 0.291 at 64; SU(4) adj
    // d_R = 15 fp64 0.347 ms at 84 with 16 sites per CTA, 0.400 with 32, 0.400 at 64 registers)
#ifndef HR_CP_REGS
#define HR_CP_REGS 84
#endif
#ifndef HR_CP_REGS_PAD   // PAD: 8 RPT accumulators + 4 RPT partial sums + one chunk of RPT x CB link elements
#define HR_CP_REGS_PAD 128
#endif
    static constexpr int REGS = PAD ? HR_CP_REGS_PAD : HR_CP_REGS * (RPT == 2 ? 3 : 2) / 2;
    // link columns per chunk of a forward hop: the whole row, or 8 when the rows are padded (two chunks of 16)
#ifndef HR_CP_CHUNK
#define HR_CP_CHUNK (PAD ? (sizeof(Real) == 8 ? 16 : 8) : D)
#endif
    static constexpr int CB = HR_CP_CHUNK;
    static_assert(LD % CB == 0 && (!PAD || CB % RPV == 0), "the chunk must divide the row and be whole vectors");
    static constexpr int MINB = 65536 / (THREADS * REGS) < 1 ? 1 : 65536 / (THREADS * REGS);
};

template <typename Real, int D, bool RL, bool MASS, bool RED>
__global__ void __launch_bounds__((CpGeom<Real, D, RL>::THREADS), (CpGeom<Real, D, RL>::MINB)) dphi_cp_kernel(const DphiArgs a)
{
    static_assert(!RED || MASS, "the fused reduction needs the self field");
    using G = CpGeom<Real, D, RL>;
    constexpr int SITES = G::SITES, RPT = G::RPT, C = G::C, EPV = G::EPV, RPV = G::RPV;
    constexpr int LNREAL = G::LNREAL_;
    constexpr int LD = G::LD, DP = G::DP;
    constexpr bool PAD = G::PAD;
    constexpr size_t LB = (size_t)LNREAL * sizeof(Real);
    // spinor entries of RPT consecutive colours form whole vectors?  (fp64: a complex IS a vector; fp32: pairs)
    constexpr bool SPIN_AL = (2 * RPT) % RPV == 0;
    // column entries (b, r0 .. r0+RPT-1) of a backward hop form whole vectors?
    constexpr bool COL_AL = RPT > 1 && (RPT * C) % RPV == 0;
    // a row of the link starts and ends on vectors?
    constexpr bool ROW_AL = EPV > 1 && D % EPV == 0;
    constexpr int EH = EPV == 1 ? LD_STREAM : LD_DEFAULT;                  // sub-vector loads go through L1
    if (a.skip != nullptr && *a.skip != 0) return;
    extern __shared__ __align__(16) unsigned char cp_smem[];
    CpPair<Real> *hs = reinterpret_cast<CpPair<Real> *>(cp_smem);          // [slot][k][b][site]

    const int sl = (int)threadIdx.x % SITES;
    const bool shadow = (int)threadIdx.x / SITES >= G::NG;
    const int r0 = (shadow ? G::NG - 1 : (int)threadIdx.x / SITES) * RPT;  // first colour row of this thread
    long s = (long)blockIdx.x * SITES + sl;
    const bool inside = s < a.vh;
    if (!inside) s = a.vh - 1;                                             // keep every thread at the barriers
    const bool live = inside && !shadow;
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

    Real acc[RPT][4][2];
#pragma unroll
    for (int rr = 0; rr < RPT; ++rr)
#pragma unroll
        for (int al = 0; al < 4; ++al) acc[rr][al][0] = acc[rr][al][1] = 0;

    // step 1 of a hop: my colours of the neighbour spinor -> my half-spinor entries -> shared memory
    auto project = [&](auto mu_c, auto dir_c, int slot, long &sn, int &sign) {
        constexpr int MU = decltype(mu_c)::value;
        constexpr int DIR = decltype(dir_c)::value;
        constexpr int S = DIR ? -1 : 1;
        constexpr int CRE = (MU == 0 || MU == 2) ? S : 0;
        constexpr int CIM = (MU == 0 || MU == 2) ? 0 : S;
        constexpr int P0 = (MU == 0 || MU == 3) ? 2 : 3;
        constexpr int P1 = 5 - P0;
        neighbour<MU, DIR>(a, g, s, sn, sign);
        Real p[4][2 * RPT];
        if constexpr (PAD) {
            // r0 is a multiple of RPV / 2 complex entries: entry al D + r0 + rr sits at a compile-time plane and half from
            // the thread's base; a dummy row (r0 + rr >= D) reads nothing and contributes zeros
            const char *inb = in + (size_t)(2 * r0 / RPV) * vh * 16;
#pragma unroll
            for (int al = 0; al < 4; ++al)
#pragma unroll
                for (int rr = 0; rr < RPT; ++rr) {
                    p[al][2 * rr] = 0; p[al][2 * rr + 1] = 0;
                    if (r0 + rr < D) load_cplx<LD_DEFAULT, 8 * D>(p[al][2 * rr], p[al][2 * rr + 1], inb, vh, (size_t)sn, al * D + rr, 0);
                }
        } else {
#pragma unroll
            for (int al = 0; al < 4; ++al) load_elems<LD_DEFAULT, 8 * D, 2, RPT, SPIN_AL>(p[al], in, vh, (size_t)sn, al * D + r0);
        }
#pragma unroll
        for (int rr = 0; rr < RPT; ++rr) {
            CpPair<Real> h0, h1;
            add_c<CRE, CIM>(h0.re, h0.im, p[0][2 * rr], p[0][2 * rr + 1], p[P0][2 * rr], p[P0][2 * rr + 1], (Real)1);
            add_c<CRE, CIM>(h1.re, h1.im, p[1][2 * rr], p[1][2 * rr + 1], p[P1][2 * rr], p[P1][2 * rr + 1], (Real)(MU >= 2 ? -1 : 1));
            hs[((slot * 2 + 0) * DP + r0 + rr) * SITES + sl] = h0;
            hs[((slot * 2 + 1) * DP + r0 + rr) * SITES + sl] = h1;
        }
    };
    // step 2: chi_{k,r} = sum_b M_{r,b} h_{k,b},  M = U(s) (forward) or U(sn)^dagger (backward); reconstruct
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
        // the link elements of this thread, ul[rr][b]: rows r0+rr of U(s) (forward) or columns r0+rr of U(sn) (backward),
        // CB columns b at a time
        constexpr int CB = G::CB;
        Real ch[RPT][4];                                                   // chi_0 (re, im), chi_1 (re, im)
#pragma unroll
        for (int rr = 0; rr < RPT; ++rr) ch[rr][0] = ch[rr][1] = ch[rr][2] = ch[rr][3] = 0;
        // PAD: per-thread bases -- rows r0.. of U start RPT * LD / RPV planes apart, columns r0.. of a row r0 / RPV planes in
        [[maybe_unused]] const char *lrow = lbase + ((size_t)(r0 * LD / RPV) * vh + ls) * 16;
        [[maybe_unused]] const char *lcol = lbase + ((size_t)(r0 / RPV) * vh + ls) * 16;
#pragma unroll
        for (int b0 = 0; b0 < LD; b0 += CB) {
            Real ul[RPT][C * CB];
            if constexpr (PAD && DIR == 0) {
#pragma unroll
                for (int rr = 0; rr < RPT; ++rr) {
#pragma unroll
                    for (int b = 0; b < CB; ++b) ul[rr][b] = 0;
                    if (r0 + rr < D) load_planes<LD_STREAM, CB / RPV>(ul[rr], lrow + (size_t)((rr * LD + b0) / RPV) * vh * 16, vh * 16, 0);
                }
            } else if constexpr (PAD) {
#pragma unroll
                for (int b = 0; b < CB; ++b) {
                    if (b0 + b >= D) continue;                               // the padding column pairs with the dummy colour: nothing to add
                    Real t[RPT];
                    load_planes<LD_STREAM, RPT / RPV>(t, lcol + (size_t)((b0 + b) * LD / RPV) * vh * 16, vh * 16, 0);
#pragma unroll
                    for (int rr = 0; rr < RPT; ++rr) ul[rr][b] = t[rr];
                }
            } else if constexpr (DIR == 0) {
#pragma unroll
                for (int rr = 0; rr < RPT; ++rr)
                    load_elems<(ROW_AL && CB == D) ? LD_STREAM : EH, LNREAL, C, CB, ROW_AL && CB == D>(ul[rr], lbase, vh, ls, (r0 + rr) * D + b0);
            } else {
#pragma unroll
                for (int b = 0; b < CB; ++b) {
                    Real t[C * RPT];
                    load_elems<COL_AL ? LD_STREAM : EH, LNREAL, C, RPT, COL_AL>(t, lbase, vh, ls, (b0 + b) * D + r0);
#pragma unroll
                    for (int rr = 0; rr < RPT; ++rr)
#pragma unroll
                        for (int c = 0; c < C; ++c) ul[rr][C * b + c] = t[C * rr + c];
                }
            }
#pragma unroll
            for (int b = 0; b < CB; ++b) {
                if (b0 + b >= D) continue;
                const CpPair<Real> h0 = hs[((slot * 2 + 0) * DP + b0 + b) * SITES + sl];
                const CpPair<Real> h1 = hs[((slot * 2 + 1) * DP + b0 + b) * SITES + sl];
#pragma unroll
                for (int rr = 0; rr < RPT; ++rr) {
                    if constexpr (RL) {
                        const Real u = ul[rr][b];
                        ch[rr][0] = fma(u, h0.re, ch[rr][0]); ch[rr][1] = fma(u, h0.im, ch[rr][1]);
                        ch[rr][2] = fma(u, h1.re, ch[rr][2]); ch[rr][3] = fma(u, h1.im, ch[rr][3]);
                    } else {
                        const Real ur = ul[rr][2 * b], ui = DIR == 1 ? -ul[rr][2 * b + 1] : ul[rr][2 * b + 1]; // backward: conj
                        ch[rr][0] = fma(ur, h0.re, ch[rr][0]); ch[rr][0] = fma(-ui, h0.im, ch[rr][0]);
                        ch[rr][1] = fma(ur, h0.im, ch[rr][1]); ch[rr][1] = fma(ui, h0.re, ch[rr][1]);
                        ch[rr][2] = fma(ur, h1.re, ch[rr][2]); ch[rr][2] = fma(-ui, h1.im, ch[rr][2]);
                        ch[rr][3] = fma(ur, h1.im, ch[rr][3]); ch[rr][3] = fma(ui, h1.re, ch[rr][3]);
                    }
                }
            }
        }
        const Real sg = (Real)sign;
        const Real sk1 = (Real)(MU >= 2 ? -1 : 1);
#pragma unroll
        for (int rr = 0; rr < RPT; ++rr) {
            acc[rr][0][0] = fma(sg, ch[rr][0], acc[rr][0][0]); acc[rr][0][1] = fma(sg, ch[rr][1], acc[rr][0][1]);
            acc_conj_c<CRE, CIM>(acc[rr][P0][0], acc[rr][P0][1], ch[rr][0], ch[rr][1], sg);
            acc[rr][1][0] = fma(sg, ch[rr][2], acc[rr][1][0]); acc[rr][1][1] = fma(sg, ch[rr][3], acc[rr][1][1]);
            acc_conj_c<CRE, CIM>(acc[rr][P1][0], acc[rr][P1][1], ch[rr][2], ch[rr][3], sg * sk1);
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

    // epilogue: my (spin, colour = r0 .. r0+RPT-1) components
    [[maybe_unused]] Real n2 = 0, dre = 0, dim = 0;
#pragma unroll
    for (int al = 0; al < 4; ++al) {
        Real o[2 * RPT];
        if constexpr (MASS) {
            Real sf[2 * RPT];
            if constexpr (PAD) {
                const char *sb = (const char *)a.self + (size_t)(2 * r0 / RPV) * vh * 16;
#pragma unroll
                for (int rr = 0; rr < RPT; ++rr) {
                    sf[2 * rr] = 0; sf[2 * rr + 1] = 0;
                    if (r0 + rr < D) load_cplx<LD_STREAM, 8 * D>(sf[2 * rr], sf[2 * rr + 1], sb, vh, (size_t)s, al * D + rr, 0);
                }
            } else load_elems<LD_STREAM, 8 * D, 2, RPT, SPIN_AL>(sf, (const char *)a.self, vh, (size_t)s, al * D + r0);
            const Real alc = coef_alpha<Real>(a, al >> 1), bec = coef_beta<Real>(a, al >> 1);
#pragma unroll
            for (int rr = 0; rr < RPT; ++rr) {
                const Real sr = sf[2 * rr], si = sf[2 * rr + 1];
                const Real orr = fma(alc, sr, bec * acc[rr][al][0]), oi = fma(alc, si, bec * acc[rr][al][1]);
                o[2 * rr] = orr; o[2 * rr + 1] = oi;
                if constexpr (RED) {
                    n2 = fma(orr, orr, fma(oi, oi, n2));
                    dre = fma(sr, orr, fma(si, oi, dre));
                    dim = fma(sr, oi, fma(-si, orr, dim));
                }
            }
        } else {
#pragma unroll
            for (int rr = 0; rr < RPT; ++rr) { o[2 * rr] = (Real)-0.5 * acc[rr][al][0]; o[2 * rr + 1] = (Real)-0.5 * acc[rr][al][1]; }
        }
        if (live) {
            const int e = al * D + r0;                                     // first complex entry
            if constexpr (PAD) {
                char *ob = (char *)a.out + ((size_t)(2 * r0 / RPV) * vh + (size_t)s) * 16;
#pragma unroll
                for (int rr = 0; rr < RPT; ++rr) {
                    if (r0 + rr >= D) continue;
                    constexpr int CPV = RPV / 2;                           // complex entries per vector
                    const int ee = al * D + rr;                            // compile-time after unrolling
                    char *q = ob + (size_t)(ee / CPV) * vh * 16 + (size_t)(ee % CPV) * (2 * sizeof(Real));
                    if constexpr (sizeof(Real) == 8) st16<ST_DEFAULT>(q, o[2 * rr], o[2 * rr + 1]);
                    else *reinterpret_cast<float2 *>(q) = make_float2((float)o[2 * rr], (float)o[2 * rr + 1]);
                }
            } else if constexpr (SPIN_AL) {
                store_planes<ST_DEFAULT, 2 * RPT / RPV>((char *)a.out + ((size_t)(2 * e / RPV) * vh + (size_t)s) * 16, vh * 16, o);
            } else {                                                       // fp32, an odd number of colours: half vectors
                static_assert(sizeof(Real) == 4, "unaligned spinor entries: fp32 only");
#pragma unroll
                for (int rr = 0; rr < RPT; ++rr)
                    *reinterpret_cast<float2 *>((char *)a.out + ((size_t)((e + rr) >> 1) * vh + (size_t)s) * 16 + (size_t)((e + rr) & 1) * 8) =
                        make_float2((float)o[2 * rr], (float)o[2 * rr + 1]);
            }
        }
    }
    if constexpr (RED) {
        double v[3] = { live ? (double)n2 : 0.0, live ? (double)dre : 0.0, live ? (double)dim : 0.0 };
        if (grid_reduce<3>(v, a.red_partial, a.red_ticket)) { a.red_result[0] = v[0]; a.red_result[1] = v[1]; a.red_result[2] = v[2]; }
    }
}

template <typename Real, int D, int LK, bool MASS, bool RED>
static hr_status launch_cp(const DphiArgs &a, cudaStream_t st)
{
    static_assert(LK == LK_COMPLEX || LK == LK_REAL, "colour-parallel kernel: represented links");
    using G = CpGeom<Real, D, LK == LK_REAL>;
    auto kern = dphi_cp_kernel<Real, D, LK == LK_REAL, MASS, RED>;
    static bool attr_set[64] = {};                   // per instantiation and device (the attribute lives in the device's context)
    int dev = 0;
    cudaGetDevice(&dev);
    if (G::smem_bytes() > 48 * 1024 && !(dev >= 0 && dev < 64 && attr_set[dev])) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::smem_bytes());
        if (e != cudaSuccess) { set_error("colour kernel: cudaFuncSetAttribute: %s", cudaGetErrorString(e)); cudaGetLastError(); return HR_ECUDA; }
        if (dev >= 0 && dev < 64) attr_set[dev] = true;
    }
    const long grid = (a.vh + G::SITES - 1) / G::SITES;
    if (RED && (unsigned long)grid > kRedMaxBlocks) { set_error("fused Dphi reduction: too many CTAs"); return HR_EUNSUPPORTED; }
    kern<<<(unsigned)grid, G::THREADS, G::smem_bytes(), st>>>(a);
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { set_error("dphi colour kernel launch failed: %s", cudaGetErrorString(e)); return HR_ECUDA; }
    return HR_OK;
}

} // namespace hr
