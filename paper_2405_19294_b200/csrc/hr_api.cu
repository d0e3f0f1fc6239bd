// hr_api.cu -- the C-ABI boundary of libhr (include/hr.h): argument checking, handles, canonical
// import/export, and the three compute calls.  Every step of the path runs in the kernels of this
// library; there is no CPU fallback (a missing/unusable CUDA device makes every compute call fail
// with HR_ECUDA).
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "hr_internal.h"

namespace hr {

static thread_local char g_err[512] = "";
static std::atomic<unsigned long long> g_launches{0};

void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}
void count_launch(int n) { g_launches.fetch_add((unsigned long long)(long long)n, std::memory_order_relaxed); }

hr_status cuda_fail(const char *what, cudaError_t e)
{
    set_error("%s: %s", what, cudaGetErrorString(e));
    return e == cudaErrorMemoryAllocation ? HR_ENOMEM : HR_ECUDA;
}
#define HR_CUDA(call)                                                                                     \
    do {                                                                                                  \
        cudaError_t e_ = (call);                                                                          \
        if (e_ != cudaSuccess) return cuda_fail(#call, e_);                                               \
    } while (0)

static int rep_dim(int N, int rep)
{
    switch (rep) {
    case HR_REP_FUND: return N;
    case HR_REP_ADJ: return N * N - 1;
    case HR_REP_SYM: return N * (N + 1) / 2;
    case HR_REP_ASYM: return N * (N - 1) / 2;
    default: return -1;
    }
}

static bool combo_supported(int N, int rep)
{
    switch (N) {
    case 2: return rep == HR_REP_FUND || rep == HR_REP_ADJ || rep == HR_REP_SYM;
    case 3: return rep == HR_REP_FUND || rep == HR_REP_ADJ || rep == HR_REP_SYM || rep == HR_REP_ASYM;
    case 4: return rep == HR_REP_FUND || rep == HR_REP_ASYM || rep == HR_REP_SYM || rep == HR_REP_ADJ;
    default: return false;
    }
}

static bool valid_prec(int p) { return p == HR_F64 || p == HR_F32; }

// is `p` device-accessible memory (device or managed)?  Host (pinned or pageable) -> false.
hr_status pointer_on_device(const void *p, bool *dev)
{
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return cuda_fail("cudaPointerGetAttributes", e);
    }
    *dev = (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged);
    return HR_OK;
}

hr_status use_device(const hr_ctx *c)
{
    cudaError_t e = cudaSetDevice(c->device);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return cuda_fail("cudaSetDevice (no usable CUDA device; libhr has no CPU fallback)", e);
    }
    return HR_OK;
}

// Staging chunk for host canonical arrays: at most this many bytes of canonical data per copy.
static const size_t kStageBytes = (size_t)256 << 20;

enum FieldKind { FIELD_GAUGE, FIELD_SPINOR };

// the context's two staging buffers, copy streams and events (first use of a host-pointer path)
static hr_status ensure_staging(hr_ctx *mc)
{
    if (mc->stage[0]) return HR_OK;
    HR_CUDA(cudaMalloc(&mc->stage[0], kStageBytes));
    cudaError_t e = cudaMalloc(&mc->stage[1], kStageBytes);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&mc->copy_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&mc->copy_stream2, cudaStreamNonBlocking);
    for (int b = 0; b < 2 && e == cudaSuccess; ++b) {
        e = cudaEventCreateWithFlags(&mc->ev_copied[b], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&mc->ev_used[b], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&mc->ev_out_ready[b], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&mc->ev_out_copied[b], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) { cudaFree(mc->stage[0]); cudaFree(mc->stage[1]); mc->stage[0] = mc->stage[1] = nullptr; return cuda_fail("staging buffers", e); }
    mc->stage_bytes = kStageBytes;
    return HR_OK;
}

// canonical (host or device) <-> internal.  `nsites_total` = sites of the canonical array
// (gauge: V full-lattice sites, 4 records each; spinor: Vh half-lattice sites of `parity`).
static hr_status transfer(const hr_ctx *c, FieldKind kind, bool import, int nreal, void *internal, hr_prec prec,
                          void *canon, hr_prec cprec, cudaStream_t st)
{
    hr_status rc = use_device(c);
    if (rc != HR_OK) return rc;
    bool dev = false;
    rc = pointer_on_device(canon, &dev);
    if (rc != HR_OK) return rc;
    const long nsites = kind == FIELD_GAUGE ? c->V : c->Vh;
    // a represented real link field with padded rows (link_ld): internal rows of ld reals, canonical rows of d_R
    const bool padded = kind == FIELD_GAUGE && link_ld(c) != c->d && nreal == c->d * link_ld(c);
    const int ld = padded ? link_ld(c) : 0, dcol = padded ? c->d : 0;
    const int cnreal = padded ? c->d * c->d : nreal;
    const size_t site_bytes = (size_t)(kind == FIELD_GAUGE ? 4 : 1) * cnreal * prec_bytes(cprec);

    auto run = [&](void *canon_dev, long first, long n) -> hr_status {
        if (kind == FIELD_GAUGE)
            return import ? launch_pack_gauge(c, nreal, ld, dcol, internal, prec, canon_dev, cprec, first, n, st)
                          : launch_unpack_gauge(c, nreal, ld, dcol, internal, prec, canon_dev, cprec, first, n, st);
        return import ? launch_pack_spinor(c, internal, prec, canon_dev, cprec, first, n, st)
                      : launch_unpack_spinor(c, internal, prec, canon_dev, cprec, first, n, st);
    };
    if (dev) return run(canon, 0, nsites);

    // host canonical array: staged through two device buffers owned by the context; the host<->device copy of one chunk
    // (copy stream) overlaps the pack / unpack kernel of the other (caller's stream); one synchronisation at the end
    // (the host array must be reusable / valid when the call returns)
    hr_ctx *mc = const_cast<hr_ctx *>(c);
    rc = ensure_staging(mc);
    if (rc != HR_OK) return rc;
    long chunk = (long)(kStageBytes / site_bytes);
    if (chunk < 1) { set_error("canonical record of %zu bytes exceeds the staging buffer", site_bytes); return HR_EUNSUPPORTED; }
    if (chunk > nsites) chunk = nsites;
    cudaStream_t cs = mc->copy_stream;
    hr_status out = HR_OK;
    cudaError_t e = cudaSuccess;
    long k = 0;
    for (long first = 0; first < nsites && out == HR_OK && e == cudaSuccess; first += chunk, ++k) {
        const long n = (nsites - first < chunk) ? nsites - first : chunk;
        const int b = (int)(k & 1);
        char *h = (char *)canon + (size_t)first * site_bytes;
        if (import) {
            if (k >= 2) e = cudaStreamWaitEvent(cs, mc->ev_used[b], 0);                 // the pack of chunk k-2 has read stage[b]
            if (e == cudaSuccess) e = cudaMemcpyAsync(mc->stage[b], h, (size_t)n * site_bytes, cudaMemcpyHostToDevice, cs);
            if (e == cudaSuccess) e = cudaEventRecord(mc->ev_copied[b], cs);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(st, mc->ev_copied[b], 0);
            if (e == cudaSuccess) out = run(mc->stage[b], first, n);
            if (e == cudaSuccess && out == HR_OK) e = cudaEventRecord(mc->ev_used[b], st);
        } else {
            if (k >= 2) e = cudaStreamWaitEvent(st, mc->ev_copied[b], 0);               // the copy of chunk k-2 has left stage[b]
            if (e == cudaSuccess) out = run(mc->stage[b], first, n);
            if (e == cudaSuccess && out == HR_OK) e = cudaEventRecord(mc->ev_used[b], st);
            if (e == cudaSuccess && out == HR_OK) e = cudaStreamWaitEvent(cs, mc->ev_used[b], 0);
            if (e == cudaSuccess && out == HR_OK) e = cudaMemcpyAsync(h, mc->stage[b], (size_t)n * site_bytes, cudaMemcpyDeviceToHost, cs);
            if (e == cudaSuccess && out == HR_OK) e = cudaEventRecord(mc->ev_copied[b], cs);
        }
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(cs);
    if (e != cudaSuccess) { cudaGetLastError(); if (out == HR_OK) out = cuda_fail("staged canonical copy", e); }
    return out;
}

} // namespace hr

using namespace hr;

extern "C" {

const char *hr_version(void) { return "hr-dphi 0.1 (sm_100a)"; }
const char *hr_last_error(void) { return g_err; }
unsigned long long hr_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

hr_status hr_ctx_create(hr_ctx **ctx, const int dims[4], const int bc[4], int N, hr_rep rep, int device)
{
    if (!ctx || !dims || !bc) { set_error("hr_ctx_create: NULL argument"); return HR_EINVAL; }
    *ctx = nullptr;
    for (int m = 0; m < 4; ++m) {
        if (dims[m] < 2 || (dims[m] & 1)) {
            set_error("hr_ctx_create: dims[%d]=%d must be even and >= 2 (reading C11)", m, dims[m]);
            return HR_EINVAL;
        }
        if (bc[m] != 1 && bc[m] != -1) { set_error("hr_ctx_create: bc[%d]=%d must be +1 or -1", m, bc[m]); return HR_EINVAL; }
    }
    if ((int)rep < 0 || (int)rep > 3) { set_error("hr_ctx_create: unknown representation %d", (int)rep); return HR_EINVAL; }
    if (device < 0) { set_error("hr_ctx_create: device=%d", device); return HR_EINVAL; }
    if (!combo_supported(N, rep)) {
        set_error("hr_ctx_create: SU(%d) representation %d is not instantiated", N, (int)rep);
        return HR_EUNSUPPORTED;
    }
    const double vol = (double)dims[0] * dims[1] * dims[2] * dims[3];
    if (vol > 2.0e9) { set_error("hr_ctx_create: volume %.3g exceeds the 2^31 index range", vol); return HR_EINVAL; }
    hr_ctx *c = new (std::nothrow) hr_ctx();
    if (!c) { set_error("hr_ctx_create: out of host memory"); return HR_ENOMEM; }
    for (int m = 0; m < 4; ++m) { c->dims[m] = dims[m]; c->bc[m] = bc[m]; }
    c->N = N;
    c->rep = (int)rep;
    c->d = rep_dim(N, rep);
    c->real_links = (rep == HR_REP_ADJ);
    c->device = device;
    c->V = (long)dims[0] * dims[1] * dims[2] * dims[3];
    c->Vh = c->V / 2;
    c->variant = -1;
    c->block = 0;
    c->xblock = 0;
    c->cg_graph = 1;
    c->bulk_rows = c->bulk_stages = c->bulk_ctas = c->bulk_strip = 0;
    c->qmr_state = nullptr;
    c->qmr_state_bytes = 0;
    c->stage[0] = c->stage[1] = nullptr;
    c->stage_bytes = 0;
    c->copy_stream = nullptr;
    c->copy_stream2 = nullptr;
    c->ws_in = c->ws_out = c->ws_stage = nullptr;
    c->ws_spinor_bytes = c->ws_stage_bytes = 0;
    c->ws_prec = -1;
    c->red_scratch = nullptr;
    c->red_scratch_bytes = 0;
    *ctx = c;
    return HR_OK;
}

void hr_ctx_destroy(hr_ctx *ctx)
{
    if (!ctx) return;
    if (ctx->ws_in || ctx->ws_out || ctx->ws_stage || ctx->red_scratch || ctx->stage[0] || ctx->qmr_state) {
        if (cudaSetDevice(ctx->device) == cudaSuccess) {
            cudaFree(ctx->qmr_state);
            if (ctx->stage[0]) {
                cudaFree(ctx->stage[0]);
                cudaFree(ctx->stage[1]);
                for (int b = 0; b < 2; ++b) {
                    cudaEventDestroy(ctx->ev_copied[b]); cudaEventDestroy(ctx->ev_used[b]);
                    cudaEventDestroy(ctx->ev_out_ready[b]); cudaEventDestroy(ctx->ev_out_copied[b]);
                }
                cudaStreamDestroy(ctx->copy_stream);
                cudaStreamDestroy(ctx->copy_stream2);
            }
            cudaFree(ctx->ws_in);
            cudaFree(ctx->ws_out);
            cudaFree(ctx->ws_stage);
            cudaFree(ctx->red_scratch);
        }
        cudaGetLastError();
    }
    delete ctx;
}

int hr_rep_dim(const hr_ctx *ctx) { return ctx ? ctx->d : -1; }
int hr_links_are_real(const hr_ctx *ctx) { return ctx ? ctx->real_links : -1; }
size_t hr_half_volume(const hr_ctx *ctx) { return ctx ? (size_t)ctx->Vh : 0; }

size_t hr_gauge_bytes(const hr_ctx *ctx, int represented, hr_prec prec)
{
    if (!ctx || !valid_prec(prec) || represented < 0 || represented > 2) return 0;
    return (size_t)ctx->V * 4 * link_nreal(ctx, represented) * prec_bytes(prec);
}

size_t hr_spinor_bytes(const hr_ctx *ctx, hr_prec prec)
{
    if (!ctx || !valid_prec(prec)) return 0;
    return (size_t)ctx->Vh * 8 * ctx->d * prec_bytes(prec);
}

hr_status hr_gauge_alloc(const hr_ctx *ctx, int represented, hr_prec prec, void *dev_mem, hr_gauge **out)
{
    if (!ctx || !out) { set_error("hr_gauge_alloc: NULL argument"); return HR_EINVAL; }
    *out = nullptr;
    if (!valid_prec(prec) || represented < 0 || represented > 2) {
        set_error("hr_gauge_alloc: bad precision or `represented` flag");
        return HR_EINVAL;
    }
    if (represented == 2 && ctx->N > 3) {
        set_error("hr_gauge_alloc: row-compressed fundamental links exist for SU(2) and SU(3) only");
        return HR_EUNSUPPORTED;
    }
    if (dev_mem && ((uintptr_t)dev_mem & 15)) { set_error("hr_gauge_alloc: dev_mem must be 16-byte aligned"); return HR_EINVAL; }
    hr_gauge *g = new (std::nothrow) hr_gauge();
    if (!g) { set_error("hr_gauge_alloc: out of host memory"); return HR_ENOMEM; }
    g->ctx = ctx;
    g->represented = represented;
    g->prec = prec;
    g->bytes = hr_gauge_bytes(ctx, represented, prec);
    g->nreal = link_nreal(ctx, represented);
    g->owns = 0;
    g->data = dev_mem;
    if (!dev_mem) {
        hr_status rc = use_device(ctx);
        if (rc != HR_OK) { delete g; return rc; }
        cudaError_t e = cudaMalloc(&g->data, g->bytes);
        if (e != cudaSuccess) { delete g; cudaGetLastError(); return cuda_fail("hr_gauge_alloc: cudaMalloc", e); }
        g->owns = 1;
    }
    *out = g;
    return HR_OK;
}

void hr_gauge_free(hr_gauge *g)
{
    if (!g) return;
    if (g->owns && g->data) {
        if (cudaSetDevice(g->ctx->device) == cudaSuccess) cudaFree(g->data);
        cudaGetLastError();
    }
    delete g;
}

void *hr_gauge_data(const hr_gauge *g) { return g ? g->data : nullptr; }

hr_status hr_gauge_import(hr_gauge *dst, const void *canon, hr_prec canon_prec, void *stream)
{
    if (!dst || !canon || !valid_prec(canon_prec)) { set_error("hr_gauge_import: bad argument"); return HR_EINVAL; }
    if (dst->represented == 2) { set_error("hr_gauge_import: a row-compressed field is filled by hr_gauge_compress"); return HR_EUNSUPPORTED; }
    return transfer(dst->ctx, FIELD_GAUGE, true, dst->nreal, dst->data, dst->prec, const_cast<void *>(canon), canon_prec,
                    (cudaStream_t)stream);
}

hr_status hr_gauge_export(const hr_gauge *src, void *canon, hr_prec canon_prec, void *stream)
{
    if (!src || !canon || !valid_prec(canon_prec)) { set_error("hr_gauge_export: bad argument"); return HR_EINVAL; }
    if (src->represented == 2) { set_error("hr_gauge_export: a row-compressed field has no canonical form; export the fundamental field"); return HR_EUNSUPPORTED; }
    return transfer(src->ctx, FIELD_GAUGE, false, src->nreal, src->data, src->prec, canon, canon_prec, (cudaStream_t)stream);
}

hr_status hr_spinor_import(const hr_ctx *ctx, void *dst_dev, hr_prec prec, const void *canon, hr_prec canon_prec,
                           int parity, void *stream)
{
    if (!ctx || !dst_dev || !canon || !valid_prec(prec) || !valid_prec(canon_prec) || (parity != 0 && parity != 1)) {
        set_error("hr_spinor_import: bad argument");
        return HR_EINVAL;
    }
    return transfer(ctx, FIELD_SPINOR, true, 8 * ctx->d, dst_dev, prec, const_cast<void *>(canon), canon_prec,
                    (cudaStream_t)stream);
}

hr_status hr_spinor_export(const hr_ctx *ctx, const void *src_dev, hr_prec prec, void *canon, hr_prec canon_prec,
                           int parity, void *stream)
{
    if (!ctx || !src_dev || !canon || !valid_prec(prec) || !valid_prec(canon_prec) || (parity != 0 && parity != 1)) {
        set_error("hr_spinor_export: bad argument");
        return HR_EINVAL;
    }
    return transfer(ctx, FIELD_SPINOR, false, 8 * ctx->d, const_cast<void *>(src_dev), prec, canon, canon_prec,
                    (cudaStream_t)stream);
}

hr_status hr_gauge_compress(hr_gauge *rows_out, const hr_gauge *fund_in, void *stream)
{
    if (!rows_out || !fund_in) { set_error("hr_gauge_compress: NULL argument"); return HR_EINVAL; }
    if (rows_out->ctx != fund_in->ctx || rows_out->represented != 2 || fund_in->represented != 0 || rows_out->prec != fund_in->prec) {
        set_error("hr_gauge_compress: need (row-compressed out, fundamental in) of one context and one precision");
        return HR_EINVAL;
    }
    hr_status rc = use_device(fund_in->ctx);
    if (rc != HR_OK) return rc;
    return launch_compress(fund_in->ctx, fund_in->prec, rows_out->data, fund_in->data, (cudaStream_t)stream);
}

hr_status hr_represent_links(hr_gauge *repr_out, const hr_gauge *fund_in, void *stream)
{
    if (!repr_out || !fund_in) { set_error("hr_represent_links: NULL argument"); return HR_EINVAL; }
    if (repr_out->ctx != fund_in->ctx) { set_error("hr_represent_links: fields belong to different contexts"); return HR_EINVAL; }
    if (repr_out->represented != 1 || fund_in->represented != 0) {
        set_error("hr_represent_links: need (represented out, fundamental in)");
        return HR_EINVAL;
    }
    if (repr_out->data == fund_in->data) { set_error("hr_represent_links: out aliases in"); return HR_EINVAL; }
    hr_status rc = use_device(fund_in->ctx);
    if (rc != HR_OK) return rc;
    return launch_represent(fund_in->ctx, fund_in->prec, fund_in->data, repr_out->prec, repr_out->data, (cudaStream_t)stream);
}

// x-block of the thread order (dphi_kernel.cuh): the largest divisor of X whose t-slice working set
// Xb*Y*Zh*(8L+2S) stays below kSliceBytes, so that +-t neighbour spinors are re-used out of L2.
// Measured (profiles/): a 25 MB slice (32^3 fp64) is re-used perfectly, a 176 MB one (64^3 fp64) is not.
static const double kSliceBytes = 32.0 * 1024 * 1024;
static int default_xblock(const hr_ctx *c, hr_prec prec)
{
    const double w = (double)prec_bytes(prec);
    const double site = 8.0 * link_nreal(c, 1) * w + 2.0 * 8 * c->d * w;
    const double row = (double)c->dims[2] * (c->dims[3] / 2) * site;
    int best = 1;
    for (int xb = 1; xb <= c->dims[1]; ++xb)
        if (c->dims[1] % xb == 0 && xb * row <= kSliceBytes) best = xb;
    return best;
}

} // extern "C"

namespace hr {
// Fill the launch arguments of one Dphi launch: out = alpha (.) self + beta (.) sum_hops, see DphiArgs.
void dphi_args(DphiArgs &a, const hr_ctx *c, void *out, const void *in, const void *self, const hr_gauge *links,
               int parity, const double alpha[2], const double beta[2])
{
    a.Xb = c->xblock > 0 ? c->xblock : default_xblock(c, links->prec);
    a.out = out;
    a.in = in;
    a.self = self;
    a.links = links->data;
    a.T = c->dims[0];
    a.X = c->dims[1];
    a.Y = c->dims[2];
    a.Zh = c->dims[3] / 2;
    a.parity = parity;
    for (int m = 0; m < 4; ++m) a.bc[m] = c->bc[m];
    a.vh = c->Vh;
    a.alpha[0] = alpha[0]; a.alpha[1] = alpha[1];
    a.beta[0] = beta[0]; a.beta[1] = beta[1];
    for (int i = 0; i < 2; ++i) { a.alphaf[i] = (float)alpha[i]; a.betaf[i] = (float)beta[i]; }
    a.red_partial = nullptr;
    a.red_ticket = nullptr;
    a.red_result = nullptr;
    a.skip = nullptr;
    a.site_mat = nullptr;
    a.site_mode = 0;
    a.t0 = 0;
    a.Tl = a.T;
    a.nsite = a.vh;
}

// Reduction scratch of the ctx: [3 * kRedMaxBlocks doubles of per-CTA partials][16 doubles of results][ticket].
hr_status get_red_scratch(hr_ctx *c, RedScratch *r, cudaStream_t st)
{
    const size_t pbytes = (size_t)3 * kRedMaxBlocks * sizeof(double);
    const size_t total = pbytes + 16 * sizeof(double) + 64;
    if (!c->red_scratch) {
        void *m = nullptr;
        cudaError_t e = cudaMalloc(&m, total);
        if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail("reduction scratch: cudaMalloc", e); }
        e = cudaMemsetAsync(m, 0, total, st);
        if (e != cudaSuccess) { cudaFree(m); return cuda_fail("reduction scratch: cudaMemsetAsync", e); }
        c->red_scratch = m;
        c->red_scratch_bytes = total;
    }
    r->partial = (double *)c->red_scratch;
    r->result = (double *)((char *)c->red_scratch + pbytes);
    r->ticket = (unsigned *)((char *)c->red_scratch + pbytes + 16 * sizeof(double));
    return HR_OK;
}
} // namespace hr

extern "C" {

hr_status hr_dphi_eo(void *out, const void *in, const hr_gauge *links, int parity, void *stream)
{
    if (!out || !in || !links) { set_error("hr_dphi_eo: NULL argument"); return HR_EINVAL; }
    if (parity != 0 && parity != 1) { set_error("hr_dphi_eo: parity=%d", parity); return HR_EINVAL; }
    if (dphi_link_kind(links->ctx, link_src(links)) < 0) {
        set_error("hr_dphi_eo: `links` must be a represented field (hr_represent_links); fundamental links are accepted "
                  "only for the fundamental and two-index representations");
        return HR_EINVAL;
    }
    if (out == in) { set_error("hr_dphi_eo: out aliases in"); return HR_EINVAL; }
    if (((uintptr_t)out | (uintptr_t)in) & 15) { set_error("hr_dphi_eo: spinor buffers must be 16-byte aligned"); return HR_EINVAL; }
    const hr_ctx *c = links->ctx;
    hr_status rc = use_device(c);
    if (rc != HR_OK) return rc;
    DphiArgs a;
    const double zero[2] = { 0.0, 0.0 }, mhalf[2] = { -0.5, -0.5 };
    dphi_args(a, c, out, in, nullptr, links, parity, zero, mhalf);
    return launch_dphi(c, links->prec, a, (cudaStream_t)stream, link_src(links));
}

hr_status hr_dirac(double m0, void *out_full, const void *in_full, const hr_gauge *links, void *stream)
{
    if (!out_full || !in_full || !links) { set_error("hr_dirac: NULL argument"); return HR_EINVAL; }
    if (dphi_link_kind(links->ctx, link_src(links)) < 0) { set_error("hr_dirac: `links` must be a represented field"); return HR_EINVAL; }
    if (out_full == in_full) { set_error("hr_dirac: out aliases in"); return HR_EINVAL; }
    if (((uintptr_t)out_full | (uintptr_t)in_full) & 15) { set_error("hr_dirac: spinor buffers must be 16-byte aligned"); return HR_EINVAL; }
    const hr_ctx *c = links->ctx;
    hr_status rc = use_device(c);
    if (rc != HR_OK) return rc;
    const size_t half = hr_spinor_bytes(c, links->prec);
    for (int p = 0; p < 2; ++p) {
        DphiArgs a;
        char *o = (char *)out_full + (size_t)p * half;
        const char *i_other = (const char *)in_full + (size_t)(1 - p) * half;
        const char *i_self = (const char *)in_full + (size_t)p * half;
        const double mass[2] = { 4.0 + m0, 4.0 + m0 }, mhalf[2] = { -0.5, -0.5 };
        dphi_args(a, c, o, i_other, i_self, links, p, mass, mhalf);
        rc = launch_dphi(c, links->prec, a, (cudaStream_t)stream, link_src(links));
        if (rc != HR_OK) return rc;
    }
    return HR_OK;
}

hr_status hr_dphi_eo_host(hr_ctx *ctx, void *out_canon, const void *in_canon, hr_prec canon_prec, const hr_gauge *links,
                          int parity, void *stream)
{
    if (!ctx || !out_canon || !in_canon || !links || !valid_prec(canon_prec)) { set_error("hr_dphi_eo_host: bad argument"); return HR_EINVAL; }
    if (links->ctx != ctx) { set_error("hr_dphi_eo_host: `links` belongs to a different context"); return HR_EINVAL; }
    if (parity != 0 && parity != 1) { set_error("hr_dphi_eo_host: parity=%d", parity); return HR_EINVAL; }
    hr_status rc = use_device(ctx);
    if (rc != HR_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t sb = hr_spinor_bytes(ctx, links->prec);
    if (ctx->ws_prec != (int)links->prec || ctx->ws_spinor_bytes != sb) {
        cudaFree(ctx->ws_in); cudaFree(ctx->ws_out);
        ctx->ws_in = ctx->ws_out = nullptr;
        ctx->ws_prec = -1;
        HR_CUDA(cudaMalloc(&ctx->ws_in, sb));
        HR_CUDA(cudaMalloc(&ctx->ws_out, sb));
        ctx->ws_spinor_bytes = sb;
        ctx->ws_prec = (int)links->prec;
    }
    bool in_dev = false, out_dev = false;
    rc = pointer_on_device(in_canon, &in_dev);
    if (rc == HR_OK) rc = pointer_on_device(out_canon, &out_dev);
    if (rc != HR_OK) return rc;
    // Host arrays on a lattice with enough time slices: a three-stream pipeline over chunks of time slices,
    //   host -> device copy of input chunk k+1  ||  pack k, Dphi_eo on the OUTPUT slices of chunk k-1, unpack  ||  device -> host
    //   copy of output chunk k-2
    // so that the two directions of the PCIe link are busy at once (PAPER.md:50 in miniature: compute what is there while the
    // rest travels).  Output chunk j needs the input chunks j-1, j, j+1 (hops in t, periodic), so chunks 1 .. C-2 follow the
    // uploads and the chunks C-1 and 0 come last.  Each staging buffer is used in halves (double buffering per direction).
    const long slice = ctx->Vh / ctx->dims[0];                                   // half-lattice sites of one time slice
    const size_t rec = (size_t)8 * ctx->d * prec_bytes(canon_prec);              // canonical bytes per site
    long ct = (long)((kStageBytes / 2) / ((size_t)slice * rec));                 // time slices per chunk
    if (ct > ctx->dims[0] / 8) ct = ctx->dims[0] / 8;
    const int T = ctx->dims[0];
    const int C = ct >= 1 ? (int)((T + ct - 1) / ct) : 0;
    if (in_dev || out_dev || C < 3 || dphi_link_kind(ctx, link_src(links)) < 0) {
        // device arrays, or a lattice too short in t: whole-field upload, one launch, whole-field download
        rc = transfer(ctx, FIELD_SPINOR, true, 8 * ctx->d, ctx->ws_in, links->prec, const_cast<void *>(in_canon), canon_prec, st);
        if (rc != HR_OK) return rc;
        rc = hr_dphi_eo(ctx->ws_out, ctx->ws_in, links, parity, stream);
        if (rc != HR_OK) return rc;
        return transfer(ctx, FIELD_SPINOR, false, 8 * ctx->d, ctx->ws_out, links->prec, out_canon, canon_prec, st);
    }
    rc = ensure_staging(ctx);
    if (rc != HR_OK) return rc;
    cudaStream_t cin = ctx->copy_stream, cout = ctx->copy_stream2;
    char *sin[2] = { (char *)ctx->stage[0], (char *)ctx->stage[0] + kStageBytes / 2 };
    char *sout[2] = { (char *)ctx->stage[1], (char *)ctx->stage[1] + kStageBytes / 2 };
    cudaError_t e = cudaSuccess;
    int nexp = 0;
    auto chunk_t0 = [&](int k) { return (int)(k * ct); };
    auto chunk_tl = [&](int k) { return (int)((k + 1) * ct <= T ? ct : T - k * ct); };
    auto import_chunk = [&](int k) -> hr_status {
        const int b = k & 1;
        const long first = (long)chunk_t0(k) * slice, n = (long)chunk_tl(k) * slice;
        if (k >= 2) e = cudaStreamWaitEvent(cin, ctx->ev_used[b], 0);               // the pack of chunk k-2 has read this half
        if (e == cudaSuccess) e = cudaMemcpyAsync(sin[b], (const char *)in_canon + (size_t)first * rec, (size_t)n * rec, cudaMemcpyHostToDevice, cin);
        if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_copied[b], cin);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ctx->ev_copied[b], 0);
        if (e != cudaSuccess) return cuda_fail("hr_dphi_eo_host: upload", e);
        hr_status r = launch_pack_spinor(ctx, ctx->ws_in, links->prec, sin[b], canon_prec, first, n, st);
        if (r == HR_OK && (e = cudaEventRecord(ctx->ev_used[b], st)) != cudaSuccess) r = cuda_fail("hr_dphi_eo_host: upload", e);
        return r;
    };
    auto compute_export = [&](int j) -> hr_status {
        const int m = nexp++ & 1;
        const long first = (long)chunk_t0(j) * slice, n = (long)chunk_tl(j) * slice;
        DphiArgs a;
        const double zero[2] = { 0.0, 0.0 }, mhalf[2] = { -0.5, -0.5 };
        dphi_args(a, ctx, ctx->ws_out, ctx->ws_in, nullptr, links, parity, zero, mhalf);
        a.t0 = chunk_t0(j); a.Tl = chunk_tl(j); a.nsite = n;
        hr_status r = launch_dphi(ctx, links->prec, a, st, link_src(links));
        if (r != HR_OK) return r;
        if (nexp > 2) e = cudaStreamWaitEvent(st, ctx->ev_out_copied[m], 0);        // the download two chunks ago has left this half
        if (e != cudaSuccess) return cuda_fail("hr_dphi_eo_host: download", e);
        r = launch_unpack_spinor(ctx, ctx->ws_out, links->prec, sout[m], canon_prec, first, n, st);
        if (r != HR_OK) return r;
        e = cudaEventRecord(ctx->ev_out_ready[m], st);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(cout, ctx->ev_out_ready[m], 0);
        if (e == cudaSuccess) e = cudaMemcpyAsync((char *)out_canon + (size_t)first * rec, sout[m], (size_t)n * rec, cudaMemcpyDeviceToHost, cout);
        if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_out_copied[m], cout);
        return e == cudaSuccess ? HR_OK : cuda_fail("hr_dphi_eo_host: download", e);
    };
    for (int k = 0; k < C && rc == HR_OK; ++k) {
        rc = import_chunk(k);
        if (rc == HR_OK && k >= 2) rc = compute_export(k - 1);
    }
    if (rc == HR_OK) rc = compute_export(C - 1);
    if (rc == HR_OK) rc = compute_export(0);
    // the host arrays must be valid / reusable when the call returns
    cudaError_t e1 = cudaStreamSynchronize(st), e2 = cudaStreamSynchronize(cin), e3 = cudaStreamSynchronize(cout);
    if (rc == HR_OK && (e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess)) {
        cudaGetLastError();
        rc = cuda_fail("hr_dphi_eo_host: pipeline", e1 != cudaSuccess ? e1 : e2 != cudaSuccess ? e2 : e3);
    }
    return rc;
}

hr_status hr_ctx_set_tuning(hr_ctx *ctx, const char *key, int value)
{
    if (!ctx || !key) { set_error("hr_ctx_set_tuning: NULL argument"); return HR_EINVAL; }
    if (!strcmp(key, "variant")) {
        if (!dphi_variant_valid(ctx, value)) { set_error("hr_ctx_set_tuning: variant %d not available for d_R=%d", value, ctx->d); return HR_EINVAL; }
        ctx->variant = value;
        return HR_OK;
    }
    if (!strcmp(key, "block")) {
        if (value < 0 || value > 1024 || (value % 32)) { set_error("hr_ctx_set_tuning: block=%d", value); return HR_EINVAL; }
        ctx->block = value;
        return HR_OK;
    }
    if (!strcmp(key, "xblock")) {
        if (value < 0 || (value > 0 && ctx->dims[1] % value)) { set_error("hr_ctx_set_tuning: xblock=%d must divide X=%d", value, ctx->dims[1]); return HR_EINVAL; }
        ctx->xblock = value;
        return HR_OK;
    }
    if (!strcmp(key, "bulk_rows") || !strcmp(key, "bulk_stages") || !strcmp(key, "bulk_ctas") || !strcmp(key, "bulk_strip")) {
        if (value < 0 || value > 128) { set_error("hr_ctx_set_tuning: %s=%d", key, value); return HR_EINVAL; }
        (key[5] == 'r' ? ctx->bulk_rows : !strcmp(key, "bulk_stages") ? ctx->bulk_stages : key[5] == 'c' ? ctx->bulk_ctas : ctx->bulk_strip) = value;
        return HR_OK;
    }
    if (!strcmp(key, "cg_graph")) {
        if (value < 0 || value > 2) { set_error("hr_ctx_set_tuning: cg_graph=%d", value); return HR_EINVAL; }
        ctx->cg_graph = value;
        return HR_OK;
    }
    set_error("hr_ctx_set_tuning: unknown key '%s'", key);
    return HR_EINVAL;
}

const char *hr_dphi_variant_name(const hr_ctx *ctx, hr_prec prec)
{
    if (!ctx || !valid_prec(prec)) return "?";
    return dphi_variant_name(ctx, prec);
}

} // extern "C"
