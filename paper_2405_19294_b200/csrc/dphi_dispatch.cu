// dphi_dispatch.cu -- run-time selection of the compiled (precision, d_R, link type) Dphi kernels.
// The paper selects N_c / representation / kernel flavour at compile time through macros
// (PAPER.md:32, :96); here every supported combination is compiled once and chosen from hr_ctx.
#include "hr_internal.h"

namespace hr {

template <typename Real, int D, bool RL>
hr_status launch_dphi_t(int variant, int block, const DphiArgs &a, cudaStream_t st);
template <typename Real, int D, bool RL> bool dphi_variant_ok_t(int variant);

static const char *const kNames[] = { "site", "site_ef", "pair", "pair_ef", "site_l1" };

// Default variant per (d_R, link type, precision, volume): filled from measurements.
static int default_variant(const hr_ctx *c, hr_prec prec)
{
    // measured on B200 (profiles/r1_variant_sweep.md): at d_R >= 6 fp64 one thread per site spills
    // and the pair kernel wins; in fp32 the whole site still fits one thread.
    if (c->d >= 6) return prec == HR_F64 ? 3 : 1;
    return 0;
}

static int resolve_variant(const hr_ctx *c, hr_prec prec) { return c->variant >= 0 ? c->variant : default_variant(c, prec); }

#define HR_COMBOS(X)                                                                                      \
    X(2, false) X(3, false) X(4, false) X(6, false) X(3, true) X(8, true)

hr_status launch_dphi(const hr_ctx *c, hr_prec prec, const DphiArgs &a, cudaStream_t st)
{
    const int v = resolve_variant(c, prec);
    const bool rl = c->real_links != 0;
#define X(D, RL)                                                                                          \
    if (c->d == D && rl == RL)                                                                            \
        return prec == HR_F64 ? launch_dphi_t<double, D, RL>(v, c->block, a, st)                         \
                              : launch_dphi_t<float, D, RL>(v, c->block, a, st);
    HR_COMBOS(X)
#undef X
    set_error("no Dphi kernel compiled for d_R=%d (%s links)", c->d, rl ? "real" : "complex");
    return HR_EUNSUPPORTED;
}

bool dphi_variant_valid(const hr_ctx *c, int variant)
{
    if (variant == -1) return true;
    const bool rl = c->real_links != 0;
#define X(D, RL)                                                                                          \
    if (c->d == D && rl == RL) return dphi_variant_ok_t<double, D, RL>(variant) || dphi_variant_ok_t<float, D, RL>(variant);
    HR_COMBOS(X)
#undef X
    return false;
}

const char *dphi_variant_name(const hr_ctx *c, hr_prec prec)
{
    const int v = resolve_variant(c, prec);
    return (v >= 0 && v < (int)(sizeof kNames / sizeof kNames[0])) ? kNames[v] : "?";
}

} // namespace hr
