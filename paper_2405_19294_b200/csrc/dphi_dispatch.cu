// dphi_dispatch.cu -- run-time selection of the compiled (precision, d_R, link type) Dphi kernels.
// The paper selects N_c / representation / kernel flavour at compile time through macros
// (PAPER.md:32, :96); here every supported combination is compiled once and chosen from hr_ctx.
#include "hr_internal.h"

namespace hr {

template <typename Real, int D, int LK>
hr_status launch_dphi_t(int variant, const LaunchTune &lt, const DphiArgs &a, cudaStream_t st);
template <typename Real, int D, int LK> bool dphi_variant_ok_t(int variant);
template <typename Real, int D, int LK> bool dphi_bulk_ok_t(const DphiArgs &a, int ks);

template <typename Real, int D, int LK> hr_status launch_halo_t(bool pack, int mu, const HaloArgs &a, cudaStream_t st);
template <typename Real, int D, int LK> hr_status launch_halo_multi_t(bool pack, const HaloArgs *a, const int *mu, int ndir, cudaStream_t st);

static const char *const kNames[] = { "site", "site_ef", "pair", "pair_ef", "site_l1", "site_pf", "colour", "bulk", "bulk2", "bulkx", "bulkx2", "site_loop" };

#define HR_COMBOS(X)                                                                                      \
    X(2, 0) X(3, 0) X(4, 0) X(6, 0) X(3, 1) X(8, 1) X(3, 2) X(6, 2) X(3, 3) X(6, 3) X(2, 4) X(3, 4) X(3, 5) X(8, 6) X(8, 7) X(10, 0) X(15, 1)

// can the bulk kernel (variants 7 / 8, ks consumer threads per site) tile this lattice?
static bool bulk_ok(const hr_ctx *c, hr_prec prec, int lk, int ks)
{
    // a persistent kernel wants several tiles per CTA: below 2^17 sites per parity (1024 tiles of 128) the defaults stay
    // with the site / colour kernels (an explicitly chosen variant 7-10 runs on any lattice it can tile)
    if (c->Vh < (1L << 17)) return false;
    DphiArgs a = {};
    a.T = c->dims[0]; a.X = c->dims[1]; a.Y = c->dims[2]; a.Zh = c->dims[3] / 2; a.vh = c->Vh;
#define X(D, LK)                                                                                          \
    if (c->d == D && lk == LK) return prec == HR_F64 ? dphi_bulk_ok_t<double, D, LK>(a, ks) : dphi_bulk_ok_t<float, D, LK>(a, ks);
    HR_COMBOS(X)
#undef X
    return false;
}

// sites of the tile the two-threads-per-site bulk kernel (variant 8) would use on this lattice: whole rows of Zh sites, a
// divisor of Y of them, at most 112 sites (dphi_bulk_kernel.cuh, bulk_geometry); 0 = none
static int bulk2_tile_sites(const hr_ctx *c)
{
    const int Y = c->dims[2], Zh = c->dims[3] / 2;
    int best = 0;
    for (int r = 1; r <= Y && r * Zh <= 112; ++r)
        if (Y % r == 0) best = r * Zh;
    return best;
}

// bulk2 where its tile fills the CTA, else bulk, else -1.  Measured (profiles/r2_staging.md, "geometry"): with 96-112 sites per
// tile (24^3 x 48: 8 rows of 12) bulk2 is 9-15 % ahead of the site kernel; on Z = 16 / 32 / 64 lattices its largest tile that
// divides Y has 64 sites -- 4 consumer warps -- and it LOSES 5-13 %, while bulk (one thread per site, 128-site tiles) is level
// with or ahead of the site kernel.
static int staged_variant(const hr_ctx *c, hr_prec prec, int lk)
{
    if (bulk2_tile_sites(c) >= 96 && bulk_ok(c, prec, lk, 2)) return 8;
    if (bulk_ok(c, prec, lk, 1)) return 7;
    return -1;
}

// Default variant per (d_R, link type, precision, volume): filled from measurements.
static int default_variant(const hr_ctx *c, hr_prec prec, int lk)
{
    // measured under sustained (power-capped) clocks, profiles/r2_staging.md: the TMA-staged kernels win where the site
    // kernel is latency-bound at its 8 warps per SM -- row-compressed links in fp64 (+5-8 %), the fp32 sextet with
    // represented links (+9 %), the fp64 sextet applied on the fly (+4 %)
    if ((lk == 4 || lk == 5) && prec == HR_F64 && bulk_ok(c, prec, lk, 1)) return 7;
    // d_R = 3 represented links in fp64 on lattices with Z <= 32 (tiles of 8 rows): +4-6 % (complex), +2 % (real) on 32^3x64,
    // 32^3x256, 64^3x32(z); on Z = 64 lattices (64^4) the site kernel stays ahead
    if ((lk == 0 || lk == 1) && c->d == 3 && prec == HR_F64 && c->dims[3] <= 32 && c->dims[3] >= 16 && bulk_ok(c, prec, lk, 1)) return 7;
    // sextet: fp64 applied on the fly, fp32 with represented links; SU(3) adjoint (real 8 x 8 links) in fp32 (24^3 x 48:
    // 0.159 -> 0.145 ms with bulk2; 32^4: 0.247 -> 0.236 ms with bulk)
    // ... and SU(4) two-index antisymmetric (d_R = 6) applied on the fly in fp64 (24^3 x 48: 0.246 -> 0.217 ms with bulk2)
    if (((lk == 2 && c->d == 6 && prec == HR_F64) || (lk == 3 && c->d == 6 && prec == HR_F64) || (lk == 0 && c->d == 6 && prec == HR_F32) ||
         (lk == 1 && c->d == 8 && prec == HR_F32))) {
        const int v = staged_variant(c, prec, lk);
        if (v >= 0) return v;
    }
    // SU(4) fundamental in fp64, Z <= 32: +1-2 % (40 x 32^3 0.291 -> 0.284 ms, 64 x 32^2 x 16 0.230 -> 0.227 ms)
    if (lk == 0 && c->d == 4 && prec == HR_F64 && c->dims[3] <= 32 && c->dims[3] >= 16 && bulk_ok(c, prec, lk, 1)) return 7;
    // on-the-fly two-index kernels hold an N x N link, not a d_R x d_R one: a whole site fits one thread
    if (lk == 2 || lk == 3 || lk == 4) return 0;
    if (lk == 6 || lk == 7) return prec == HR_F64 ? 2 : 0; // fp64 d_R = 8: two threads per site (measured)
    if (lk == 5) return 1;
    // d_R > 8 (SU(4) sym / adj): a site no longer fits a thread at all -- the colour-parallel kernel
    if (c->d > 8) return 6;
    // measured on B200 (profiles/r1_variant_sweep.md): at d_R >= 6 fp64 one thread per site spills
    // and the pair kernel wins; in fp32 the whole site still fits one thread.
    // ... and (bench_large_n, profiles/r1_large_n.md) the colour-parallel kernel beats both: SU(3) sextet 24^3x48 fp64
    // 0.301 ms against 0.331 (site) / 0.332 (pair); SU(3) adjoint 0.347 against 0.363 (pair_ef)
    if (c->d >= 6) return prec == HR_F64 ? 6 : 1;
    // SU(2) adjoint (real 3x3 links, spinors are 40 % of the compulsory bytes): evict-first links / evict-last
    // spinors gain 2 % (0.0965 -> 0.0944 ms at 32^4 fp64)
    if (lk == 1 && c->d == 3) return 1;
    return 0;
}

static int resolve_variant(const hr_ctx *c, hr_prec prec, int lk) { return c->variant >= 0 ? c->variant : default_variant(c, prec, lk); }
// the variant for a launch that carries a fused site matrix: the staged kernels have no such epilogue, so where one of
// them is the DEFAULT the site kernel it replaced takes these launches (an explicitly chosen variant is respected)
static int resolve_variant_fused(const hr_ctx *c, hr_prec prec, int lk)
{
    const int v = resolve_variant(c, prec, lk);
    if (c->variant < 0 && v >= 7) return (lk == 1 && c->d == 3) ? 1 : 0;
    return v;
}

// link kind (dphi_kernel.cuh): 0 complex d_R x d_R, 1 real d_R x d_R (adjoint), 2 / 3 two-index symmetric /
// antisymmetric applied on the fly from the fundamental link
int dphi_link_kind(const hr_ctx *c, int link_src)
{
    if (link_src == 0) return c->real_links ? 1 : 0;
    if (link_src == 1) {                                   // full fundamental field
        if (c->rep == HR_REP_FUND) return 0;               // FUND: both fields are N x N complex
        if (c->rep == HR_REP_SYM) return 2;
        if (c->rep == HR_REP_ASYM) return 3;
        if (c->rep == HR_REP_ADJ && c->N == 3) return 6;   // SU(3) adjoint on the fly
        return -1;                                         // SU(2) adjoint: from the row-compressed field (kind 5)
    }
    if (c->N > 3) return -1;                               // rows: SU(2), SU(3)
    if (c->rep == HR_REP_FUND) return 4;
    if (c->rep == HR_REP_ADJ && c->N == 2) return 5;
    if (c->rep == HR_REP_ADJ && c->N == 3) return 7;
    return -1;
}

hr_status launch_dphi(const hr_ctx *c, hr_prec prec, const DphiArgs &a, cudaStream_t st, int link_src)
{
    const int lk = dphi_link_kind(c, link_src);
    if (lk < 0) {
        set_error("this kind of link field has no kernel for this representation (use hr_represent_links)");
        return HR_EUNSUPPORTED;
    }
    int v = a.site_mode != 0 ? resolve_variant_fused(c, prec, lk) : resolve_variant(c, prec, lk);
    // a launch over a range of time slices (hr_dphi_eo_host's pipeline): the one-thread-per-site kernels take it
    if (a.Tl != a.T && v != 0 && v != 1) v = (lk == 1 && c->d == 3) ? 1 : 0;
    const LaunchTune lt = { c->block, c->bulk_rows, c->bulk_stages, c->bulk_ctas, c->bulk_strip };
#define X(D, LK)                                                                                          \
    if (c->d == D && lk == LK)                                                                            \
        return prec == HR_F64 ? launch_dphi_t<double, D, LK>(v, lt, a, st)                               \
                              : launch_dphi_t<float, D, LK>(v, lt, a, st);
    HR_COMBOS(X)
#undef X
    set_error("no Dphi kernel compiled for d_R=%d (link kind %d)", c->d, lk);
    return HR_EUNSUPPORTED;
}

hr_status launch_halo(const hr_ctx *c, hr_prec prec, bool pack, int mu, const HaloArgs &a, cudaStream_t st, int link_src)
{
    const int lk = dphi_link_kind(c, link_src);
#define X(D, LK)                                                                                          \
    if (c->d == D && lk == LK)                                                                            \
        return prec == HR_F64 ? launch_halo_t<double, D, LK>(pack, mu, a, st) : launch_halo_t<float, D, LK>(pack, mu, a, st);
    HR_COMBOS(X)
#undef X
    set_error("no halo kernel compiled for d_R=%d (link kind %d)", c->d, lk);
    return HR_EUNSUPPORTED;
}

hr_status launch_halo_multi(const hr_ctx *c, hr_prec prec, bool pack, const HaloArgs *a, const int *mu, int ndir, cudaStream_t st, int link_src)
{
    const int lk = dphi_link_kind(c, link_src);
#define X(D, LK)                                                                                          \
    if (c->d == D && lk == LK)                                                                            \
        return prec == HR_F64 ? launch_halo_multi_t<double, D, LK>(pack, a, mu, ndir, st) : launch_halo_multi_t<float, D, LK>(pack, a, mu, ndir, st);
    HR_COMBOS(X)
#undef X
    set_error("no halo kernel compiled for d_R=%d (link kind %d)", c->d, lk);
    return HR_EUNSUPPORTED;
}

// can a launch with this link source carry a fused site matrix (DphiArgs::site_mode)?
bool dphi_site_fusable(const hr_ctx *c, hr_prec prec, int link_src)
{
    const int lk = dphi_link_kind(c, link_src);
    // measured: fp64 d_R = 3 gains 18-30 %; fp32 (128-register cap) is no faster fused, and at
    // d_R >= 6 the block mat-vec spills in a kernel already at 255 registers
    if ((lk != 0 && lk != 1) || c->d > 4 || prec != HR_F64) return false;
    const int v = resolve_variant_fused(c, prec, lk);
    return v == 0 || v == 1;
}

bool dphi_variant_valid(const hr_ctx *c, int variant)
{
    if (variant == -1) return true;
    const int lk = c->real_links ? 1 : 0;
#define X(D, LK)                                                                                          \
    if (c->d == D && lk == LK) return dphi_variant_ok_t<double, D, LK>(variant) || dphi_variant_ok_t<float, D, LK>(variant);
    HR_COMBOS(X)
#undef X
    return false;
}

const char *dphi_variant_name(const hr_ctx *c, hr_prec prec)
{
    const int v = resolve_variant(c, prec, c->real_links ? 1 : 0);
    return (v >= 0 && v < (int)(sizeof kNames / sizeof kNames[0])) ? kNames[v] : "?";
}

} // namespace hr
