// hr_api_clover.cu -- C-ABI entry points of SURVEY.md section 8(f) NEXT-4 (include/hr.h, fourth part): the clover
// term.  Argument checking and launch sequencing only; the arithmetic is in clover.cu and the Dphi kernels.
#include "hr_internal.h"

using namespace hr;

static bool aligned16(const void *p) { return ((uintptr_t)p & 15) == 0; }

extern "C" {

size_t hr_clover_bytes(const hr_ctx *ctx, hr_prec prec)
{
    if (!ctx || (prec != HR_F64 && prec != HR_F32)) return 0;
    return (size_t)ctx->V * clover_nreal(ctx) * prec_bytes(prec);
}

hr_status hr_clover_build(void *clover, const hr_gauge *links, double csw, void *stream)
{
    if (!clover || !links) { set_error("hr_clover_build: NULL argument"); return HR_EINVAL; }
    if (links->represented != 1) { set_error("hr_clover_build: `links` must be a represented field (the leaves are products of U^R)"); return HR_EINVAL; }
    if (!aligned16(clover)) { set_error("hr_clover_build: buffer must be 16-byte aligned"); return HR_EINVAL; }
    hr_status rc = use_device(links->ctx);
    if (rc != HR_OK) return rc;
    return launch_clover_build(links->ctx, links->prec, clover, links->data, csw, (cudaStream_t)stream);
}

hr_status hr_clover_exp(const hr_ctx *ctx, hr_prec prec, void *clover, double m0, void *stream)
{
    if (!ctx || !clover || (prec != HR_F64 && prec != HR_F32)) { set_error("hr_clover_exp: bad argument"); return HR_EINVAL; }
    if (!aligned16(clover)) { set_error("hr_clover_exp: buffer must be 16-byte aligned"); return HR_EINVAL; }
    if (!(4.0 + m0 > 0.0)) { set_error("hr_clover_exp: 4 + m0 = %g must be positive", 4.0 + m0); return HR_EINVAL; }
    hr_status rc = use_device(ctx);
    if (rc != HR_OK) return rc;
    return launch_clover_exp(ctx, prec, clover, 4.0 + m0, (cudaStream_t)stream);
}

hr_status hr_dirac_clover(double m0, void *out_full, const void *in_full, const hr_gauge *links, const void *clover, void *stream)
{
    if (!out_full || !in_full || !links || !clover) { set_error("hr_dirac_clover: NULL argument"); return HR_EINVAL; }
    if (out_full == in_full) { set_error("hr_dirac_clover: out aliases in"); return HR_EINVAL; }
    if (!aligned16(out_full) || !aligned16(in_full) || !aligned16(clover)) { set_error("hr_dirac_clover: buffers must be 16-byte aligned"); return HR_EINVAL; }
    const hr_ctx *c = links->ctx;
    const size_t half = (size_t)c->Vh * 8 * c->d * prec_bytes(links->prec);
    const size_t chalf = (size_t)c->Vh * clover_nreal(c) * prec_bytes(links->prec);
    hr_status rc;
    if (links->represented == 1 && dphi_site_fusable(c, links->prec, link_src(links))) {
        // T psi fused into the Dphi epilogue: one launch per parity, nothing else touches the fields
        rc = use_device(c);
        if (rc != HR_OK) return rc;
        const double mass[2] = { 4.0 + m0, 4.0 + m0 }, mhalf[2] = { -0.5, -0.5 };
        for (int p = 0; p < 2; ++p) {
            DphiArgs a;
            dphi_args(a, c, (char *)out_full + p * half, (const char *)in_full + (1 - p) * half, (const char *)in_full + p * half,
                      links, p, mass, mhalf);
            a.site_mat = (const char *)clover + p * chalf;
            a.site_mode = 1;
            rc = launch_dphi(c, links->prec, a, (cudaStream_t)stream, link_src(links));
            if (rc != HR_OK) return rc;
        }
        return HR_OK;
    }
    rc = hr_dirac(m0, out_full, in_full, links, stream);   // (4+m0) psi + Dphi psi, two launches
    if (rc != HR_OK) return rc;
    for (int p = 0; p < 2; ++p) {                                     // out_p += T in_p
        rc = launch_clover_apply(c, links->prec, (char *)out_full + p * half, (const char *)in_full + p * half,
                                 (const char *)clover + p * chalf, (cudaStream_t)stream);
        if (rc != HR_OK) return rc;
    }
    return HR_OK;
}

} // extern "C"
