// hr_api_solver.cu -- C-ABI entry points of the rows SURVEY.md section 8(f) NEXT-1 adds (include/hr.h,
// second part): spinor linear algebra, the even-odd preconditioned operator Dhat, and the CG / full solve
// built on them.  Argument checking and launch sequencing only; the arithmetic is in linalg.cu, cg.cu and
// the Dphi kernels.  No CPU fallback.
#include <cmath>
#include <cstring>
#include <functional>

#include "hr_internal.h"

using namespace hr;

#define HR_CUDA(call)                                                                                     \
    do {                                                                                                  \
        cudaError_t e_ = (call);                                                                          \
        if (e_ != cudaSuccess) return cuda_fail(#call, e_);                                               \
    } while (0)

static bool valid_prec(int p) { return p == HR_F64 || p == HR_F32; }
static bool aligned16(const void *p) { return ((uintptr_t)p & 15) == 0; }

// copy `n` doubles of a device result to `dst`, which may be host (synchronises) or device memory
static hr_status deliver(double *dst, const double *src_dev, int n, cudaStream_t st)
{
    bool dev = false;
    hr_status rc = pointer_on_device(dst, &dev);
    if (rc != HR_OK) return rc;
    HR_CUDA(cudaMemcpyAsync(dst, src_dev, (size_t)n * sizeof(double), dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, st));
    if (!dev) HR_CUDA(cudaStreamSynchronize(st));
    return HR_OK;
}

// tmp_o = Dphi_oe in ; out = [gamma5] (m^2 in - Dphi_eo tmp_o).  red != null: also reduce |out|^2, <in,out>.
static hr_status dhat_launches(const hr_ctx *c, double m0, int g5, void *out_e, const void *in_e, void *tmp_o,
                               const hr_gauge *links, const RedScratch *rs, double *red_result, const int *skip,
                               cudaStream_t st)
{
    const double m = 4.0 + m0;
    const double zero[2] = { 0.0, 0.0 }, mhalf[2] = { -0.5, -0.5 };
    DphiArgs a;
    dphi_args(a, c, tmp_o, in_e, nullptr, links, 1, zero, mhalf);
    a.skip = skip;
    hr_status rc = launch_dphi(c, links->prec, a, st, link_src(links));
    if (rc != HR_OK) return rc;
    const double s = g5 ? -1.0 : 1.0;
    const double alpha[2] = { m * m, s * m * m }, beta[2] = { 0.5, s * 0.5 }; // -Dphi = +1/2 sum_hops
    dphi_args(a, c, out_e, tmp_o, in_e, links, 0, alpha, beta);
    a.skip = skip;
    if (rs) {
        a.red_partial = rs->partial;
        a.red_ticket = rs->ticket;
        a.red_result = red_result;
    }
    return launch_dphi(c, links->prec, a, st, link_src(links));
}

extern "C" {

hr_status hr_spinor_lincomb(const hr_ctx *ctx, hr_prec prec, void *out, const double ca[2], int g5, const void *x,
                            const double cb[2], const void *y, void *stream)
{
    if (!ctx || !out || !x || !ca || !valid_prec(prec) || (y && !cb)) { set_error("hr_spinor_lincomb: bad argument"); return HR_EINVAL; }
    if (!aligned16(out) || !aligned16(x) || !aligned16(y)) { set_error("hr_spinor_lincomb: buffers must be 16-byte aligned"); return HR_EINVAL; }
    hr_status rc = use_device(ctx);
    if (rc != HR_OK) return rc;
    const double zero[2] = { 0.0, 0.0 };
    return launch_lincomb(ctx, prec, out, ca, g5 != 0, x, y ? cb : zero, y, (cudaStream_t)stream);
}

hr_status hr_spinor_copy(const hr_ctx *ctx, hr_prec prec, void *out, const void *in, void *stream)
{
    const double one[2] = { 1.0, 0.0 };
    return hr_spinor_lincomb(ctx, prec, out, one, 0, in, nullptr, nullptr, stream);
}

hr_status hr_spinor_g5(const hr_ctx *ctx, hr_prec prec, void *out, const void *in, void *stream)
{
    const double one[2] = { 1.0, 0.0 };
    return hr_spinor_lincomb(ctx, prec, out, one, 1, in, nullptr, nullptr, stream);
}

hr_status hr_spinor_mulc_add_assign(const hr_ctx *ctx, hr_prec prec, void *out, double c_re, double c_im, const void *in,
                                    void *stream)
{
    const double c[2] = { c_re, c_im }, one[2] = { 1.0, 0.0 };
    return hr_spinor_lincomb(ctx, prec, out, c, 0, in, one, out, stream);
}

hr_status hr_spinor_g5_mulc_add_assign(const hr_ctx *ctx, hr_prec prec, void *out, double c_re, double c_im, const void *in,
                                       void *stream)
{
    const double c[2] = { c_re, c_im }, one[2] = { 1.0, 0.0 };
    return hr_spinor_lincomb(ctx, prec, out, c, 1, in, one, out, stream);
}

hr_status hr_spinor_dot(hr_ctx *ctx, hr_prec prec, const void *x, const void *y, double *result, void *stream)
{
    if (!ctx || !x || !y || !result || !valid_prec(prec)) { set_error("hr_spinor_dot: bad argument"); return HR_EINVAL; }
    if (!aligned16(x) || !aligned16(y)) { set_error("hr_spinor_dot: buffers must be 16-byte aligned"); return HR_EINVAL; }
    hr_status rc = use_device(ctx);
    if (rc != HR_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    RedScratch rs;
    rc = get_red_scratch(ctx, &rs, st);
    if (rc != HR_OK) return rc;
    rc = launch_dot(ctx, prec, x, y, rs, rs.result, st);
    if (rc != HR_OK) return rc;
    return deliver(result, rs.result, 2, st);
}

hr_status hr_spinor_norm2(hr_ctx *ctx, hr_prec prec, const void *x, double *result, void *stream)
{
    if (!ctx || !x || !result || !valid_prec(prec)) { set_error("hr_spinor_norm2: bad argument"); return HR_EINVAL; }
    if (!aligned16(x)) { set_error("hr_spinor_norm2: buffer must be 16-byte aligned"); return HR_EINVAL; }
    hr_status rc = use_device(ctx);
    if (rc != HR_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    RedScratch rs;
    rc = get_red_scratch(ctx, &rs, st);
    if (rc != HR_OK) return rc;
    rc = launch_dot(ctx, prec, x, x, rs, rs.result, st);
    if (rc != HR_OK) return rc;
    return deliver(result, rs.result, 1, st);
}

hr_status hr_dhat(double m0, int g5, void *out_e, const void *in_e, void *tmp_o, const hr_gauge *links, void *stream)
{
    if (!out_e || !in_e || !tmp_o || !links) { set_error("hr_dhat: NULL argument"); return HR_EINVAL; }
    if (dphi_link_kind(links->ctx, link_src(links)) < 0) { set_error("hr_dhat: `links` must be a represented field"); return HR_EINVAL; }
    if (out_e == in_e || out_e == tmp_o || in_e == tmp_o) { set_error("hr_dhat: out, in and tmp must be distinct buffers"); return HR_EINVAL; }
    if (!aligned16(out_e) || !aligned16(in_e) || !aligned16(tmp_o)) { set_error("hr_dhat: buffers must be 16-byte aligned"); return HR_EINVAL; }
    const hr_ctx *c = links->ctx;
    hr_status rc = use_device(c);
    if (rc != HR_OK) return rc;
    return dhat_launches(c, m0, g5 != 0, out_e, in_e, tmp_o, links, nullptr, nullptr, nullptr, (cudaStream_t)stream);
}

size_t hr_cg_workspace_bytes(const hr_ctx *ctx, hr_prec prec, int maxiter)
{
    if (!ctx || !valid_prec(prec) || maxiter < 0) return 0;
    const size_t sb = (size_t)ctx->Vh * 8 * ctx->d * prec_bytes(prec);
    const size_t state = (sizeof(CgState) + ((size_t)maxiter + 2) * sizeof(double) + 255) & ~(size_t)255;
    return 5 * sb + state;
}

// CG on (gamma5 Dhat)^2 x = rhs with rhs already in ws.r; see hr.h
static hr_status cg_run(hr_ctx *c, double m0, void *x_e, const hr_gauge *links, double tol, int maxiter, char *ws,
                        int *iters, double *rel_res2, double *hist_host, cudaStream_t st)
{
    const hr_prec prec = links->prec;
    const size_t sb = (size_t)c->Vh * 8 * c->d * prec_bytes(prec);
    void *r = ws, *p = ws + sb, *t = ws + 2 * sb, *ap = ws + 3 * sb, *tmp = ws + 4 * sb;
    CgState *cs = (CgState *)(ws + 5 * sb);
    RedScratch rs;
    hr_status rc = get_red_scratch(c, &rs, st);
    if (rc != HR_OK) return rc;
    rc = launch_cg_init(c, prec, cs, tol, maxiter, x_e, p, r, rs, st);
    if (rc != HR_OK) return rc;
    CgState h;
    memset(&h, 0, sizeof h);
    auto one_iteration = [&](cudaStream_t q) -> hr_status {
        hr_status e = dhat_launches(c, m0, 1, t, p, tmp, links, &rs, &cs->pap, &cs->done, q);   // t = Q p, pap = |Q p|^2
        if (e != HR_OK) return e;
        e = dhat_launches(c, m0, 1, ap, t, tmp, links, nullptr, nullptr, &cs->done, q);         // Ap = Q t
        if (e != HR_OK) return e;
        e = launch_cg_update_r(c, prec, cs, r, ap, rs, q);
        if (e != HR_OK) return e;
        return launch_cg_update_xp(c, prec, cs, x_e, p, r, q);
    };
    // Nothing in an iteration changes from the host's point of view (alpha, beta, k and the stop flags are on the
    // device), so ONE iteration is captured into a CUDA graph once and replayed: 6 kernel launches cost one graph
    // launch -- what matters on the small local lattices of a strong-scaling run, where the paper finds the
    // time "dominated by the kernel call overheads".  Captured on a private stream (the caller's
    // may be the legacy default stream, which cannot capture); falls back to plain launches if capture fails.
    // Measured on B200: -13 % per iteration at 8^4 (41 -> 35 us), -8 % at 32 x 16^3, nothing to
    // gain once an iteration takes a millisecond: cg_graph = 1 replays below 2^19 sites per parity, 2 always.
    cudaGraphExec_t gexec = nullptr;
    if (c->cg_graph == 2 || (c->cg_graph == 1 && c->Vh <= (1L << 19))) {
        cudaStream_t cap = nullptr;
        cudaGraph_t graph = nullptr;
        const unsigned long long before = hr_launch_count();
        bool ok = cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking) == cudaSuccess;
        if (ok) ok = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
        if (ok) {
            const hr_status e = one_iteration(cap);
            const cudaError_t ce = cudaStreamEndCapture(cap, &graph);
            ok = e == HR_OK && ce == cudaSuccess && graph != nullptr;
        }
        if (ok) ok = cudaGraphInstantiate(&gexec, graph, 0) == cudaSuccess;
        if (graph) cudaGraphDestroy(graph);
        if (cap) cudaStreamDestroy(cap);
        count_launch(-(int)(hr_launch_count() - before)); // captured, not launched
        if (!ok) { gexec = nullptr; cudaGetLastError(); }
    }
    // iterations are enqueued in batches; the host looks at the device state once per batch.  A batch
    // that overshoots costs only empty launches (every kernel returns at once when `done` is set).
    int batch = 4;
    rc = HR_OK;
    for (int issued = 0; rc == HR_OK;) {
        cudaError_t ce = cudaMemcpyAsync(&h, cs, sizeof h, cudaMemcpyDeviceToHost, st);
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
        if (ce != cudaSuccess) { rc = cuda_fail("CG state read-back", ce); break; }
        if (h.done || issued >= maxiter) break;
        int n = maxiter - issued < batch ? maxiter - issued : batch;
        for (int i = 0; i < n && rc == HR_OK; ++i) {
            if (gexec) {
                ce = cudaGraphLaunch(gexec, st);
                if (ce != cudaSuccess) rc = cuda_fail("cudaGraphLaunch (CG iteration)", ce);
                else count_launch(6);
            } else {
                rc = one_iteration(st);
            }
        }
        issued += n;
        if (batch < 32) batch *= 2;
    }
    if (gexec) cudaGraphExecDestroy(gexec);
    if (rc != HR_OK) return rc;
    if (iters) *iters = h.iter;
    if (rel_res2 || hist_host) {
        const int n = h.iter + 1;
        if (hist_host) {
            HR_CUDA(cudaMemcpyAsync(hist_host, (const double *)(cs + 1), (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, st));
            HR_CUDA(cudaStreamSynchronize(st));
            if (rel_res2) *rel_res2 = h.bb > 0 ? hist_host[h.iter] / h.bb : 0.0;
            if (h.bb > 0) for (int k = 0; k < n; ++k) hist_host[k] /= h.bb;
        } else {
            double last = 0;
            HR_CUDA(cudaMemcpyAsync(&last, (const double *)(cs + 1) + h.iter, sizeof(double), cudaMemcpyDeviceToHost, st));
            HR_CUDA(cudaStreamSynchronize(st));
            *rel_res2 = h.bb > 0 ? last / h.bb : 0.0;
        }
    }
    return HR_OK;
}

static hr_status cg_check(const char *who, hr_ctx *ctx, const void *x, const void *b, const hr_gauge *links, double tol,
                          int maxiter, const void *ws)
{
    if (!ctx || !x || !b || !links || !ws) { set_error("%s: NULL argument", who); return HR_EINVAL; }
    if (links->ctx != ctx) { set_error("%s: `links` belongs to a different context", who); return HR_EINVAL; }
    if (dphi_link_kind(ctx, link_src(links)) < 0) { set_error("%s: `links` must be a represented field", who); return HR_EINVAL; }
    if (!(tol >= 0.0) || maxiter < 0) { set_error("%s: tol=%g maxiter=%d", who, tol, maxiter); return HR_EINVAL; }
    if (x == b) { set_error("%s: x aliases b", who); return HR_EINVAL; }
    if (!aligned16(x) || !aligned16(b) || ((uintptr_t)ws & 255)) { set_error("%s: buffers must be 16-byte (workspace 256-byte) aligned", who); return HR_EINVAL; }
    return use_device(ctx);
}

hr_status hr_cg_dhat(hr_ctx *ctx, double m0, void *x_e, const void *b_e, const hr_gauge *links, double tol, int maxiter,
                     void *workspace, int *iters, double *rel_res2, double *hist, void *stream)
{
    hr_status rc = cg_check("hr_cg_dhat", ctx, x_e, b_e, links, tol, maxiter, workspace);
    if (rc != HR_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    char *ws = (char *)workspace;
    const size_t sb = (size_t)ctx->Vh * 8 * ctx->d * prec_bytes(links->prec);
    // rhs = Dhat^dagger b = Q gamma5 b  (reading C21): t = gamma5 b ; r = Q t
    const double one[2] = { 1.0, 0.0 }, zero[2] = { 0.0, 0.0 };
    rc = launch_lincomb(ctx, links->prec, ws + 2 * sb, one, 1, b_e, zero, nullptr, st);
    if (rc != HR_OK) return rc;
    rc = dhat_launches(ctx, m0, 1, ws, ws + 2 * sb, ws + 4 * sb, links, nullptr, nullptr, nullptr, st);
    if (rc != HR_OK) return rc;
    return cg_run(ctx, m0, x_e, links, tol, maxiter, ws, iters, rel_res2, hist, st);
}

size_t hr_cg_dist_workspace_bytes(const hr_ctx *ctx, hr_prec prec)
{
    if (!ctx || !valid_prec(prec)) return 0;
    const size_t sb = ((size_t)ctx->Vh * 8 * ctx->d * prec_bytes(prec) + 255) & ~(size_t)255;
    return 6 * sb;   // r, p, Ap, w, tmp_o, tmp_e
}

// CG on Dhat^dagger Dhat = (gamma5 Dhat)^2 with the operator's two Dphi_eo and the cross-rank sums supplied by the caller;
// everything else -- vector updates, scalar recurrences, stopping test -- is done here (oracle/solver.py::cg_dhat, step by step)
hr_status hr_cg_dhat_dist(hr_ctx *ctx, hr_prec prec, double m0, void *x_e, const void *b_e, double tol, int maxiter,
                          void *workspace, hr_dphi_fn dphi, hr_allsum_fn allsum, void *user, int *iters, double *hist,
                          void *stream)
{
    if (!ctx || !x_e || !b_e || !workspace || !dphi || !valid_prec(prec) || maxiter < 0 || !(tol >= 0)) {
        set_error("hr_cg_dhat_dist: bad argument");
        return HR_EINVAL;
    }
    if (x_e == b_e || !aligned16(x_e) || !aligned16(b_e) || ((uintptr_t)workspace & 255)) {
        set_error("hr_cg_dhat_dist: x aliases b, or a buffer is misaligned (fields 16, workspace 256 bytes)");
        return HR_EINVAL;
    }
    hr_status rc = use_device(ctx);
    if (rc != HR_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    RedScratch rs;
    rc = get_red_scratch(ctx, &rs, st);
    if (rc != HR_OK) return rc;
    const size_t sb = ((size_t)ctx->Vh * 8 * ctx->d * prec_bytes(prec) + 255) & ~(size_t)255;
    char *ws = (char *)workspace;
    void *r = ws, *p = ws + sb, *ap = ws + 2 * sb, *w = ws + 3 * sb, *tmp_o = ws + 4 * sb, *tmp_e = ws + 5 * sb;
    const double m = 4.0 + m0, one[2] = { 1, 0 }, zero[2] = { 0, 0 }, mm[2] = { m * m, 0 }, minus[2] = { -1, 0 };

    auto cb_fail = [&](const char *what) { set_error("hr_cg_dhat_dist: the %s callback failed", what); return HR_ECUDA; };
    // out = gamma5 Dhat in,  Dhat = (4+m0)^2 - Dphi_eo Dphi_oe
    auto g5dhat = [&](void *out, const void *in) -> hr_status {
        if (dphi(user, tmp_o, in, 1) != 0) return cb_fail("dphi");
        if (dphi(user, tmp_e, tmp_o, 0) != 0) return cb_fail("dphi");
        hr_status q = launch_lincomb(ctx, prec, tmp_e, mm, 0, in, minus, tmp_e, st);
        if (q != HR_OK) return q;
        return launch_lincomb(ctx, prec, out, one, 1, tmp_e, zero, nullptr, st);
    };
    // global sum over the ranks of the local <a, b> (real part) -- |a|^2 when a == b
    auto gdot = [&](const void *a, const void *b, double *out) -> hr_status {
        hr_status q = launch_dot(ctx, prec, a, b, rs, rs.result, st);
        if (q != HR_OK) return q;
        double v[2];
        q = deliver(v, rs.result, 2, st);
        if (q != HR_OK) return q;
        if (allsum && allsum(user, v, 1) != 0) return cb_fail("allsum");
        *out = v[0];
        return HR_OK;
    };
#define HR_TRY(x) do { hr_status q_ = (x); if (q_ != HR_OK) return q_; } while (0)
    // rhs = Dhat^dagger b = gamma5 Dhat gamma5 b;  x = 0, r = p = rhs
    HR_TRY(launch_lincomb(ctx, prec, w, one, 1, b_e, zero, nullptr, st));
    HR_TRY(g5dhat(r, w));
    HR_TRY(launch_lincomb(ctx, prec, p, one, 0, r, zero, nullptr, st));
    HR_TRY(launch_lincomb(ctx, prec, x_e, zero, 0, r, zero, nullptr, st));
    double bb = 0;
    HR_TRY(gdot(r, r, &bb));
    double rr = bb;
    int k = 0;
    if (hist) hist[0] = bb > 0 ? 1.0 : 0.0;
    while (bb > 0 && k < maxiter && rr > tol * tol * bb) {
        HR_TRY(g5dhat(w, p));
        HR_TRY(g5dhat(ap, w));
        double pap = 0;
        HR_TRY(gdot(p, ap, &pap));
        const double alpha = rr / pap;
        const double pa[2] = { alpha, 0 }, na[2] = { -alpha, 0 };
        HR_TRY(launch_lincomb(ctx, prec, x_e, one, 0, x_e, pa, p, st));
        HR_TRY(launch_lincomb(ctx, prec, r, one, 0, r, na, ap, st));
        double rr_new = 0;
        HR_TRY(gdot(r, r, &rr_new));
        const double beta[2] = { rr_new / rr, 0 };
        HR_TRY(launch_lincomb(ctx, prec, p, one, 0, r, beta, p, st));
        rr = rr_new;
        ++k;
        if (hist) hist[k] = rr / bb;
    }
#undef HR_TRY
    if (iters) *iters = k;
    return HR_OK;
}

size_t hr_bicgstab_workspace_bytes(const hr_ctx *ctx, hr_prec prec, int maxiter)
{
    if (!ctx || !valid_prec(prec) || maxiter < 0) return 0;
    return 7 * (size_t)ctx->Vh * 8 * ctx->d * prec_bytes(prec) + bicgstab_state_bytes(maxiter);
}

} // extern "C"

// The operator of a BiCGstab run: out = Op in.  reduce: also leave |out|^2 and <in, out> in red[0..2] (the Dphi
// epilogue does it for Dhat; operators that end in another kernel use two dot launches).  skip: device flag, non-zero =
// converged (kernels that know about it return at once).
typedef std::function<hr_status(void *out, const void *in, bool reduce, double *red, const int *skip, cudaStream_t q)> BiOp;

// textbook BiCGstab on device-resident scalars (bicgstab.cu); ws holds r, rhat, p, v, s, t (6 half spinors) and the state
static hr_status bicgstab_core(hr_ctx *ctx, hr_prec prec, void *x_e, const void *b_e, double tol, int maxiter, char *ws,
                               void *state, const BiOp &op, int *iters, double *rel_res2, double *hist, cudaStream_t st)
{
    const size_t sb = (size_t)ctx->Vh * 8 * ctx->d * prec_bytes(prec);
    void *r = ws, *rhat = ws + sb, *p = ws + 2 * sb, *v = ws + 3 * sb, *s = ws + 4 * sb, *t = ws + 5 * sb;
    RedScratch rs;
    hr_status rc = get_red_scratch(ctx, &rs, st);
    if (rc != HR_OK) return rc;
    rc = launch_bi_init(ctx, prec, state, tol, maxiter, x_e, r, rhat, p, v, b_e, rs, st);
    if (rc != HR_OK) return rc;
    const int *done = bicgstab_done(state);
    auto one_iteration = [&](cudaStream_t q) -> hr_status {
        hr_status e = launch_bi_update_p(ctx, prec, state, p, r, v, q);
        if (e != HR_OK) return e;
        e = op(v, p, false, nullptr, done, q);                                                               // v = Op p
        if (e != HR_OK) return e;
        e = launch_dot(ctx, prec, rhat, v, rs, bicgstab_rhat_v(state), q);                                  // <rhat, v>
        if (e != HR_OK) return e;
        e = launch_bi_update_s(ctx, prec, state, s, r, v, q);
        if (e != HR_OK) return e;
        e = op(t, s, true, bicgstab_tt_st(state), done, q);                                                 // t = Op s, |t|^2, <s,t>
        if (e != HR_OK) return e;
        return launch_bi_update_xr(ctx, prec, state, x_e, r, p, s, t, rhat, rs, q);
    };
    // as in the CG: an iteration is host-invariant, so on small lattices it is captured once and replayed as a graph
    cudaGraphExec_t gexec = nullptr;
    int launches_per_iteration = 0;
    if (ctx->cg_graph == 2 || (ctx->cg_graph == 1 && ctx->Vh <= (1L << 19))) {
        cudaStream_t cap = nullptr;
        cudaGraph_t graph = nullptr;
        const unsigned long long before = hr_launch_count();
        bool ok = cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking) == cudaSuccess;
        if (ok) ok = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
        if (ok) {
            const hr_status e = one_iteration(cap);
            const cudaError_t ce = cudaStreamEndCapture(cap, &graph);
            ok = e == HR_OK && ce == cudaSuccess && graph != nullptr;
        }
        if (ok) ok = cudaGraphInstantiate(&gexec, graph, 0) == cudaSuccess;
        if (graph) cudaGraphDestroy(graph);
        if (cap) cudaStreamDestroy(cap);
        launches_per_iteration = (int)(hr_launch_count() - before);
        count_launch(-launches_per_iteration); // captured, not launched
        if (!ok) { gexec = nullptr; cudaGetLastError(); }
    }
    alignas(8) char hbuf[256];
    const size_t hb = bicgstab_header_bytes();
    int it = 0, dn = 0;
    double bb = 0;
    int batch = 4;
    for (int issued = 0;;) {
        HR_CUDA(cudaMemcpyAsync(hbuf, state, hb, cudaMemcpyDeviceToHost, st));
        HR_CUDA(cudaStreamSynchronize(st));
        bicgstab_unpack(hbuf, &it, &dn, &bb);
        if (dn || issued >= maxiter) break;
        const int n = maxiter - issued < batch ? maxiter - issued : batch;
        for (int i = 0; i < n; ++i) {
            if (gexec) {
                const cudaError_t ce = cudaGraphLaunch(gexec, st);
                if (ce != cudaSuccess) { cudaGraphExecDestroy(gexec); return cuda_fail("cudaGraphLaunch (BiCGstab iteration)", ce); }
                count_launch(launches_per_iteration);
            } else {
                rc = one_iteration(st);
                if (rc != HR_OK) return rc;
            }
        }
        issued += n;
        if (batch < 32) batch *= 2;
    }
    if (gexec) cudaGraphExecDestroy(gexec);
    if (iters) *iters = it;
    const double *dh = (const double *)((const char *)state + hb);
    if (hist) {
        HR_CUDA(cudaMemcpyAsync(hist, dh, (size_t)(it + 1) * sizeof(double), cudaMemcpyDeviceToHost, st));
        HR_CUDA(cudaStreamSynchronize(st));
        if (rel_res2) *rel_res2 = bb > 0 ? hist[it] / bb : 0.0;
        if (bb > 0) for (int k = 0; k <= it; ++k) hist[k] /= bb;
    } else if (rel_res2) {
        double last = 0;
        HR_CUDA(cudaMemcpyAsync(&last, dh + it, sizeof(double), cudaMemcpyDeviceToHost, st));
        HR_CUDA(cudaStreamSynchronize(st));
        *rel_res2 = bb > 0 ? last / bb : 0.0;
    }
    return HR_OK;
}

// Dhat_sw = A_ee - Dphi_eo A_oo^{-1} Dphi_oe (reading C32): 2 Dphi launches + 2 site-local launches
static hr_status dhat_clover_launches(const hr_ctx *c, void *out_e, const void *in_e, void *tmp_o, void *tmp2_o,
                                      const hr_gauge *links, const void *site, const void *site_inv, const int *skip, cudaStream_t st)
{
    const size_t chalf = (size_t)c->Vh * clover_nreal(c) * prec_bytes(links->prec);
    const double zero[2] = { 0.0, 0.0 }, mhalf[2] = { -0.5, -0.5 }, phalf[2] = { 0.5, 0.5 };
    DphiArgs a;
    if (links->represented == 1 && dphi_site_fusable(c, links->prec, link_src(links))) {
        // both site-local steps fused into the Dphi epilogues: tmp2 = A_oo^{-1} (Dphi_oe in); out = A_ee in - Dphi_eo tmp2
        dphi_args(a, c, tmp2_o, in_e, nullptr, links, 1, zero, mhalf);
        a.skip = skip;
        a.site_mat = (const char *)site_inv + chalf;
        a.site_mode = 2;
        hr_status rc = launch_dphi(c, links->prec, a, st, link_src(links));
        if (rc != HR_OK) return rc;
        dphi_args(a, c, out_e, tmp2_o, in_e, links, 0, zero, phalf);     // 0 * in + 1/2 hops (= -Dphi) + A_ee in
        a.skip = skip;
        a.site_mat = site;
        a.site_mode = 1;
        return launch_dphi(c, links->prec, a, st, link_src(links));
    }
    dphi_args(a, c, tmp_o, in_e, nullptr, links, 1, zero, mhalf);
    a.skip = skip;
    hr_status rc = launch_dphi(c, links->prec, a, st, link_src(links));                                     // tmp = Dphi_oe in
    if (rc != HR_OK) return rc;
    rc = launch_clover_apply(c, links->prec, tmp2_o, tmp_o, (const char *)site_inv + chalf, st, 0);        // tmp2 = A_oo^{-1} tmp
    if (rc != HR_OK) return rc;
    dphi_args(a, c, out_e, tmp2_o, nullptr, links, 0, zero, mhalf);
    a.skip = skip;
    rc = launch_dphi(c, links->prec, a, st, link_src(links));                                               // out = Dphi_eo tmp2
    if (rc != HR_OK) return rc;
    return launch_clover_apply(c, links->prec, out_e, in_e, site, st, -1);                                  // out = A_ee in - out
}

extern "C" {

hr_status hr_bicgstab_dhat(hr_ctx *ctx, double m0, void *x_e, const void *b_e, const hr_gauge *links, double tol, int maxiter,
                           void *workspace, int *iters, double *rel_res2, double *hist, void *stream)
{
    hr_status rc = cg_check("hr_bicgstab_dhat", ctx, x_e, b_e, links, tol, maxiter, workspace);
    if (rc != HR_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    char *ws = (char *)workspace;
    const size_t sb = (size_t)ctx->Vh * 8 * ctx->d * prec_bytes(links->prec);
    void *tmp = ws + 6 * sb;
    RedScratch rs;
    rc = get_red_scratch(ctx, &rs, st);
    if (rc != HR_OK) return rc;
    BiOp op = [&](void *out, const void *in, bool reduce, double *red, const int *skip, cudaStream_t q) -> hr_status {
        return dhat_launches(ctx, m0, 0, out, in, tmp, links, reduce ? &rs : nullptr, red, skip, q);
    };
    return bicgstab_core(ctx, links->prec, x_e, b_e, tol, maxiter, ws, ws + 7 * sb, op, iters, rel_res2, hist, st);
}

size_t hr_qmr_workspace_bytes(const hr_ctx *ctx, hr_prec prec)
{
    if (!ctx || !valid_prec(prec)) return 0;
    return 6 * (size_t)ctx->Vh * 8 * ctx->d * prec_bytes(prec);
}

// gamma5-QMR on Dhat (include/hr.h; reading C33).  Host-driven: the Lanczos scalars and the Givens rotations live on the
// host, two stream synchronisations per iteration; every vector operation is a library kernel.
hr_status hr_qmr_dhat(hr_ctx *ctx, double m0, void *x_e, const void *b_e, const hr_gauge *links, double tol, int maxiter,
                      void *workspace, int *iters, double *rel_res2, double *hist, void *stream)
{
    hr_status rc = cg_check("hr_qmr_dhat", ctx, x_e, b_e, links, tol, maxiter, workspace);
    if (rc != HR_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const hr_prec P = links->prec;
    const size_t sb = (size_t)ctx->Vh * 8 * ctx->d * prec_bytes(P);
    const size_t nvec = sb / 16, half = nvec / 2;
    char *ws = (char *)workspace;
    void *v = ws, *vp = ws + sb, *p1 = ws + 2 * sb, *p2 = ws + 3 * sb, *w = ws + 4 * sb, *tmp = ws + 5 * sb;
    RedScratch rs;
    rc = get_red_scratch(ctx, &rs, st);
    if (rc != HR_OK) return rc;
    const double zero[2] = { 0.0, 0.0 }, one[2] = { 1.0, 0.0 };
    double h[8];
    // |x_upper|^2 and |x_lower|^2 of a field: its norm and its gamma5 "norm" <x, gamma5 x> in one read each half
    auto halves = [&](const void *f, double *up, double *lo) -> hr_status {
        hr_status r = launch_dot_range(ctx, P, f, f, 0, half, rs, rs.result, st);
        if (r != HR_OK) return r;
        r = launch_dot_range(ctx, P, f, f, half, half, rs, rs.result + 2, st);
        if (r != HR_OK) return r;
        HR_CUDA(cudaMemcpyAsync(h, rs.result, 4 * sizeof(double), cudaMemcpyDeviceToHost, st));
        HR_CUDA(cudaStreamSynchronize(st));
        *up = h[0]; *lo = h[2];
        return HR_OK;
    };
    auto true_res2 = [&](double bb, double *out) -> hr_status {      // |b - Dhat x|^2 / |b|^2, through w and tmp
        hr_status r = dhat_launches(ctx, m0, 0, w, x_e, tmp, links, nullptr, nullptr, nullptr, st);
        if (r != HR_OK) return r;
        const double m1[2] = { -1.0, 0.0 };
        r = launch_lincomb(ctx, P, w, one, 0, b_e, m1, w, st);
        if (r != HR_OK) return r;
        double up, lo;
        r = halves(w, &up, &lo);
        if (r != HR_OK) return r;
        *out = (up + lo) / bb;
        return HR_OK;
    };
    rc = launch_lincomb(ctx, P, x_e, zero, 0, b_e, zero, nullptr, st);                    // x = 0
    if (rc != HR_OK) return rc;
    double up, lo;
    rc = halves(b_e, &up, &lo);
    if (rc != HR_OK) return rc;
    const double bb = up + lo, bnorm = sqrt(bb);
    if (hist) hist[0] = bb > 0.0 ? 1.0 : 0.0;
    if (iters) *iters = 0;
    if (rel_res2) *rel_res2 = bb > 0.0 ? 1.0 : 0.0;
    if (bb == 0.0) return HR_OK;
    // the device-resident state (Lanczos scalars, rotations, history): owned by the context, grown with maxiter
    const size_t need = (sizeof(QmrState) + ((size_t)maxiter + 2) * sizeof(double) + 255) & ~(size_t)255;
    if (ctx->qmr_state_bytes < need) {
        if (ctx->qmr_state) { HR_CUDA(cudaStreamSynchronize(st)); cudaFree(ctx->qmr_state); ctx->qmr_state = nullptr; ctx->qmr_state_bytes = 0; }
        HR_CUDA(cudaMalloc(&ctx->qmr_state, need));
        ctx->qmr_state_bytes = need;
    }
    QmrState *qs = (QmrState *)ctx->qmr_state;
    const double inv[2] = { 1.0 / bnorm, 0.0 };
    // buffers by iteration parity: v_k in va (k even) / vb (k odd), v_{k-1} in the other; p_{k-1} in pa (k even) / pb, p_{k-2} in the other
    void *va = v, *vb = vp, *pa = p1, *pb = p2;
    rc = launch_lincomb(ctx, P, va, inv, 0, b_e, zero, nullptr, st);                      // v_1 = b / rho_1
    if (rc != HR_OK) return rc;
    rc = launch_lincomb(ctx, P, pa, zero, 0, b_e, zero, nullptr, st);                     // p_0 = p_{-1} = 0
    if (rc != HR_OK) return rc;
    rc = launch_lincomb(ctx, P, pb, zero, 0, b_e, zero, nullptr, st);
    if (rc != HR_OK) return rc;
    rc = launch_qmr_init(qs, bnorm, (up - lo) / bb, tol, maxiter, st);
    if (rc != HR_OK) return rc;
    // one iteration, with the buffer roles of iteration index kk: 2 Dphi launches (fused reduction -> (v, Dhat v)_J), the
    // Lanczos kernel, the update kernel and two one-thread kernels for the scalar recurrences -- nothing returns to the host
    auto enqueue = [&](int kk) -> hr_status {
        void *vk = (kk & 1) ? vb : va, *vprev = (kk & 1) ? va : vb;
        void *pk1 = (kk & 1) ? pb : pa, *pk2 = (kk & 1) ? pa : pb;
        hr_status r = dhat_launches(ctx, m0, 1, w, vk, tmp, links, &rs, qs->red + 4, &qs->stop, st);   // w = gamma5 Dhat v
        if (r != HR_OK) return r;
        r = launch_qmr_scal_a(qs, st);
        if (r != HR_OK) return r;
        r = launch_qmr_lanczos(ctx, P, w, vk, vprev, qs, rs, st);    // vt = gamma5 w - alpha v - beta v_prev (into w) + its half norms
        if (r != HR_OK) return r;
        r = launch_qmr_scal_b(qs, st);
        if (r != HR_OK) return r;
        // p = (v - eps p_{k-1} - theta p_{k-2}) / zeta into p_{k-2}'s buffer; x += c eta p; v_{k+1} = vt / rho_{k+1} into v_{k-1}'s buffer
        return launch_qmr_update(ctx, P, pk2, pk1, vk, x_e, vprev, w, qs, st);
    };
    QmrState hs;
    double res2 = 1.0;
    bool have_res = false;
    int k = 0, batch = 4;
    for (;;) {
        const int n = maxiter - k < batch ? maxiter - k : batch;
        for (int j = 0; j < n; ++j) { rc = enqueue(k + j); if (rc != HR_OK) return rc; }
        HR_CUDA(cudaMemcpyAsync(&hs, qs, sizeof(QmrState), cudaMemcpyDeviceToHost, st));
        HR_CUDA(cudaStreamSynchronize(st));
        k = hs.k;
        if (hs.stop == 1) {                                   // quasi-residual below tol: the TRUE residual decides
            rc = true_res2(bb, &res2);
            if (rc != HR_OK) return rc;
            have_res = true;
            if (res2 <= tol * tol || k >= maxiter) break;
            have_res = false;
            rc = launch_qmr_resume(qs, st);
            if (rc != HR_OK) return rc;
            if (k >= maxiter) break;
            continue;
        }
        if (hs.stop != 0 || k >= maxiter) break;
        if (batch < 32) batch *= 2;
    }
    if (!have_res) { rc = true_res2(bb, &res2); if (rc != HR_OK) return rc; }
    if (hist && k > 0) HR_CUDA(cudaMemcpy(hist + 1, reinterpret_cast<const double *>(qs + 1) + 1, (size_t)k * sizeof(double), cudaMemcpyDeviceToHost));
    if (iters) *iters = k;
    if (rel_res2) *rel_res2 = res2;
    return HR_OK;
}

hr_status hr_clover_finalize(const hr_ctx *ctx, hr_prec prec, void *site_term, void *site_inverse, double m0, void *stream)
{
    if (!ctx || !site_term || !site_inverse || !valid_prec(prec) || site_term == site_inverse) { set_error("hr_clover_finalize: bad argument"); return HR_EINVAL; }
    if (!aligned16(site_term) || !aligned16(site_inverse)) { set_error("hr_clover_finalize: buffers must be 16-byte aligned"); return HR_EINVAL; }
    hr_status rc = use_device(ctx);
    if (rc != HR_OK) return rc;
    return launch_clover_finalize(ctx, prec, site_term, site_inverse, 4.0 + m0, (cudaStream_t)stream);
}

hr_status hr_dhat_clover(void *out_e, const void *in_e, void *tmp_o, void *tmp2_o, const hr_gauge *links, const void *site_term,
                         const void *site_inverse, void *stream)
{
    if (!out_e || !in_e || !tmp_o || !tmp2_o || !links || !site_term || !site_inverse) { set_error("hr_dhat_clover: NULL argument"); return HR_EINVAL; }
    if (dphi_link_kind(links->ctx, link_src(links)) < 0) { set_error("hr_dhat_clover: no kernel for this kind of link field"); return HR_EINVAL; }
    if (out_e == in_e || out_e == tmp_o || out_e == tmp2_o || in_e == tmp_o || in_e == tmp2_o || tmp_o == tmp2_o) {
        set_error("hr_dhat_clover: out, in and the two temporaries must be distinct buffers");
        return HR_EINVAL;
    }
    if (!aligned16(out_e) || !aligned16(in_e) || !aligned16(tmp_o) || !aligned16(tmp2_o) || !aligned16(site_term) || !aligned16(site_inverse)) {
        set_error("hr_dhat_clover: buffers must be 16-byte aligned");
        return HR_EINVAL;
    }
    hr_status rc = use_device(links->ctx);
    if (rc != HR_OK) return rc;
    return dhat_clover_launches(links->ctx, out_e, in_e, tmp_o, tmp2_o, links, site_term, site_inverse, nullptr, (cudaStream_t)stream);
}

size_t hr_clover_solve_workspace_bytes(const hr_ctx *ctx, hr_prec prec, int maxiter)
{
    if (!ctx || !valid_prec(prec) || maxiter < 0) return 0;
    return 8 * (size_t)ctx->Vh * 8 * ctx->d * prec_bytes(prec) + bicgstab_state_bytes(maxiter);
}

hr_status hr_dirac_clover_solve(hr_ctx *ctx, void *x_full, const void *b_full, const hr_gauge *links, const void *site_term,
                                const void *site_inverse, double tol, int maxiter, void *workspace, int *iters, double *rel_res2,
                                void *stream)
{
    hr_status rc = cg_check("hr_dirac_clover_solve", ctx, x_full, b_full, links, tol, maxiter, workspace);
    if (rc != HR_OK) return rc;
    if (!site_term || !site_inverse || !aligned16(site_term) || !aligned16(site_inverse)) { set_error("hr_dirac_clover_solve: bad site-term buffers"); return HR_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    const hr_prec prec = links->prec;
    char *ws = (char *)workspace;
    const size_t sb = (size_t)ctx->Vh * 8 * ctx->d * prec_bytes(prec);
    const size_t chalf = (size_t)ctx->Vh * clover_nreal(ctx) * prec_bytes(prec);
    void *tmp = ws + 6 * sb, *tmp2 = ws + 7 * sb, *state = ws + 8 * sb;
    char *x_e = (char *)x_full, *x_o = (char *)x_full + sb;
    const char *b_e = (const char *)b_full, *b_o = (const char *)b_full + sb;
    const char *ainv_o = (const char *)site_inverse + chalf;
    const double zero[2] = { 0.0, 0.0 }, mhalf[2] = { -0.5, -0.5 }, one[2] = { 1.0, 0.0 }, mone[2] = { -1.0, 0.0 };
    RedScratch rs;
    rc = get_red_scratch(ctx, &rs, st);
    if (rc != HR_OK) return rc;
    // reading C32: bhat = b_e - Dphi_eo A_oo^{-1} b_o, kept in the x_o slot until the end
    rc = launch_clover_apply(ctx, prec, tmp2, b_o, ainv_o, st, 0);
    if (rc != HR_OK) return rc;
    DphiArgs a;
    dphi_args(a, ctx, x_o, tmp2, nullptr, links, 0, zero, mhalf);
    rc = launch_dphi(ctx, prec, a, st, link_src(links));
    if (rc != HR_OK) return rc;
    rc = launch_lincomb(ctx, prec, x_o, one, 0, b_e, mone, x_o, st);
    if (rc != HR_OK) return rc;
    BiOp op = [&](void *out, const void *in, bool reduce, double *red, const int *skip, cudaStream_t q) -> hr_status {
        hr_status e = dhat_clover_launches(ctx, out, in, tmp, tmp2, links, site_term, site_inverse, skip, q);
        if (e != HR_OK || !reduce) return e;
        e = launch_dot(ctx, prec, out, out, rs, red, q);           // red[0] = |out|^2 (red[1] = 0, overwritten next)
        if (e != HR_OK) return e;
        return launch_dot(ctx, prec, in, out, rs, red + 1, q);     // red[1..2] = <in, out>
    };
    rc = bicgstab_core(ctx, prec, x_e, x_o, tol, maxiter, ws, state, op, iters, rel_res2, nullptr, st);
    if (rc != HR_OK) return rc;
    // x_o = A_oo^{-1} (b_o - Dphi_oe x_e)
    dphi_args(a, ctx, tmp, x_e, nullptr, links, 1, zero, mhalf);
    rc = launch_dphi(ctx, prec, a, st, link_src(links));
    if (rc != HR_OK) return rc;
    rc = launch_lincomb(ctx, prec, tmp, one, 0, b_o, mone, tmp, st);
    if (rc != HR_OK) return rc;
    return launch_clover_apply(ctx, prec, x_o, tmp, ainv_o, st, 0);
}

hr_status hr_dirac_solve(hr_ctx *ctx, double m0, void *x_full, const void *b_full, const hr_gauge *links, double tol,
                         int maxiter, void *workspace, int *iters, double *rel_res2, void *stream)
{
    hr_status rc = cg_check("hr_dirac_solve", ctx, x_full, b_full, links, tol, maxiter, workspace);
    if (rc != HR_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const hr_prec prec = links->prec;
    char *ws = (char *)workspace;
    const size_t sb = (size_t)ctx->Vh * 8 * ctx->d * prec_bytes(prec);
    const double m = 4.0 + m0;
    char *x_e = (char *)x_full, *x_o = (char *)x_full + sb;
    const char *b_e = (const char *)b_full, *b_o = (const char *)b_full + sb;
    // reading C24:  bhat = m b_e - Dphi_eo b_o  (kept in the x_o slot until the end)
    DphiArgs a;
    const double am[2] = { m, m }, half[2] = { 0.5, 0.5 };
    dphi_args(a, ctx, x_o, b_o, b_e, links, 0, am, half);
    rc = launch_dphi(ctx, prec, a, st, link_src(links));
    if (rc != HR_OK) return rc;
    // rhs of the normal equations: r = Q gamma5 bhat
    const double one[2] = { 1.0, 0.0 }, zero[2] = { 0.0, 0.0 };
    rc = launch_lincomb(ctx, prec, ws + 2 * sb, one, 1, x_o, zero, nullptr, st);
    if (rc != HR_OK) return rc;
    rc = dhat_launches(ctx, m0, 1, ws, ws + 2 * sb, ws + 4 * sb, links, nullptr, nullptr, nullptr, st);
    if (rc != HR_OK) return rc;
    rc = cg_run(ctx, m0, x_e, links, tol, maxiter, ws, iters, rel_res2, nullptr, st);
    if (rc != HR_OK) return rc;
    // x_o = (b_o - Dphi_oe x_e) / m
    const double ainv[2] = { 1.0 / m, 1.0 / m }, binv[2] = { 0.5 / m, 0.5 / m };
    dphi_args(a, ctx, x_o, x_e, b_o, links, 1, ainv, binv);
    return launch_dphi(ctx, prec, a, st, link_src(links));
}

hr_status hr_dirac_solve_bicgstab(hr_ctx *ctx, double m0, void *x_full, const void *b_full, const hr_gauge *links, double tol,
                                  int maxiter, void *workspace, int *iters, double *rel_res2, void *stream)
{
    hr_status rc = cg_check("hr_dirac_solve_bicgstab", ctx, x_full, b_full, links, tol, maxiter, workspace);
    if (rc != HR_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const hr_prec prec = links->prec;
    const size_t sb = (size_t)ctx->Vh * 8 * ctx->d * prec_bytes(prec);
    const double m = 4.0 + m0;
    char *x_e = (char *)x_full, *x_o = (char *)x_full + sb;
    const char *b_e = (const char *)b_full, *b_o = (const char *)b_full + sb;
    // reading C24:  bhat = m b_e - Dphi_eo b_o  (kept in the x_o slot until the end); BiCGstab on Dhat x_e = bhat
    DphiArgs a;
    const double am[2] = { m, m }, half[2] = { 0.5, 0.5 };
    dphi_args(a, ctx, x_o, b_o, b_e, links, 0, am, half);
    rc = launch_dphi(ctx, prec, a, st, link_src(links));
    if (rc != HR_OK) return rc;
    rc = hr_bicgstab_dhat(ctx, m0, x_e, x_o, links, tol, maxiter, workspace, iters, rel_res2, nullptr, stream);
    if (rc != HR_OK) return rc;
    const double ainv[2] = { 1.0 / m, 1.0 / m }, binv[2] = { 0.5 / m, 0.5 / m };
    dphi_args(a, ctx, x_o, x_e, b_o, links, 1, ainv, binv);
    return launch_dphi(ctx, prec, a, st, link_src(links));
}

size_t hr_mixed_workspace_bytes(const hr_ctx *ctx, int maxiter)
{
    if (!ctx || maxiter < 0) return 0;
    const size_t s64 = (size_t)ctx->Vh * 8 * ctx->d * 8, s32 = s64 / 2;
    return 3 * s64 + 2 * s32 + hr_bicgstab_workspace_bytes(ctx, HR_F32, maxiter);
}

hr_status hr_bicgstab_dhat_mixed(hr_ctx *ctx, double m0, void *x_e, const void *b_e, const hr_gauge *links64,
                                 const hr_gauge *links32, double tol, double inner_tol, int maxiter, void *workspace,
                                 int *iters, int *outer_steps, double *rel_res2, void *stream)
{
    hr_status rc = cg_check("hr_bicgstab_dhat_mixed", ctx, x_e, b_e, links64, tol, maxiter, workspace);
    if (rc != HR_OK) return rc;
    if (!links32 || links32->ctx != ctx || links64->prec != HR_F64 || links32->prec != HR_F32 ||
        dphi_link_kind(ctx, link_src(links32)) < 0 || !(inner_tol > 0.0 && inner_tol < 1.0)) {
        set_error("hr_bicgstab_dhat_mixed: need an fp64 and an fp32 link field of this context and 0 < inner_tol < 1");
        return HR_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    char *ws = (char *)workspace;
    const size_t s64 = (size_t)ctx->Vh * 8 * ctx->d * 8, s32 = s64 / 2;
    void *r = ws, *ax = ws + s64, *tmp = ws + 2 * s64, *r32 = ws + 3 * s64, *e32 = ws + 3 * s64 + s32;
    void *inner_ws = ws + 3 * s64 + 2 * s32;
    const double one[2] = { 1.0, 0.0 }, zero[2] = { 0.0, 0.0 }, mone[2] = { -1.0, 0.0 };
    RedScratch rs;
    rc = get_red_scratch(ctx, &rs, st);
    if (rc != HR_OK) return rc;
    // x = 0, r = b
    rc = launch_lincomb(ctx, HR_F64, x_e, zero, 0, b_e, zero, nullptr, st);
    if (rc != HR_OK) return rc;
    rc = launch_lincomb(ctx, HR_F64, r, one, 0, b_e, zero, nullptr, st);
    if (rc != HR_OK) return rc;
    double bb = -1.0, rr = 0.0;
    int total = 0, outer = 0;
    for (;;) {
        rc = launch_dot(ctx, HR_F64, r, r, rs, rs.result, st);
        if (rc != HR_OK) return rc;
        HR_CUDA(cudaMemcpyAsync(&rr, rs.result, sizeof(double), cudaMemcpyDeviceToHost, st));
        HR_CUDA(cudaStreamSynchronize(st));
        if (bb < 0) bb = rr;
        if (!(rr > tol * tol * bb) || total >= maxiter || outer >= 100) break;
        // defect equation Dhat e = r, solved in fp32 on the normalised residual
        const double nrm = sqrt(rr);
        rc = launch_cvt(ctx, true, r32, r, 1.0 / nrm, st);
        if (rc != HR_OK) return rc;
        int it = 0;
        rc = hr_bicgstab_dhat(ctx, m0, e32, r32, links32, inner_tol, maxiter - total, inner_ws, &it, nullptr, nullptr, stream);
        if (rc != HR_OK) return rc;
        total += it;
        ++outer;
        rc = launch_cvt(ctx, false, x_e, e32, nrm, st);                                               // x += |r| e
        if (rc != HR_OK) return rc;
        rc = dhat_launches(ctx, m0, 0, ax, x_e, tmp, links64, nullptr, nullptr, nullptr, st);         // fp64 true residual
        if (rc != HR_OK) return rc;
        rc = launch_lincomb(ctx, HR_F64, r, one, 0, b_e, mone, ax, st);                               // r = b - Dhat x
        if (rc != HR_OK) return rc;
        if (it == 0) {                                                                                // no progress possible:
            rc = launch_dot(ctx, HR_F64, r, r, rs, rs.result, st);                                    // report the residual of
            if (rc != HR_OK) return rc;                                                               // the x that is returned
            HR_CUDA(cudaMemcpyAsync(&rr, rs.result, sizeof(double), cudaMemcpyDeviceToHost, st));
            HR_CUDA(cudaStreamSynchronize(st));
            break;
        }
    }
    if (iters) *iters = total;
    if (outer_steps) *outer_steps = outer;
    if (rel_res2) *rel_res2 = bb > 0 ? rr / bb : 0.0;
    return HR_OK;
}

} // extern "C"
