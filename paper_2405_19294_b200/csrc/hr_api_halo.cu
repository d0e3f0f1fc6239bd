// hr_api_halo.cu -- C-ABI entry points of SURVEY.md section 8(e)/(f) NEXT-2 (include/hr.h, third part):
// Dphi_eo on a lattice split into slabs along t, one slab per GPU, half-spinor messages.
// Argument checking and launch sequencing only; the arithmetic is in halo_kernel.cuh and dphi_kernel.cuh.
#include <cstring>

#include "hr_internal.h"

using namespace hr;

static bool aligned16(const void *p) { return ((uintptr_t)p & 15) == 0; }

static hr_status check_links(const char *who, const hr_gauge *links, int parity)
{
    if (!links) { set_error("%s: NULL links", who); return HR_EINVAL; }
    if (parity != 0 && parity != 1) { set_error("%s: parity=%d", who, parity); return HR_EINVAL; }
    if (dphi_link_kind(links->ctx, link_src(links)) < 0) {
        set_error("%s: `links` must be a represented field for this representation", who);
        return HR_EINVAL;
    }
    return use_device(links->ctx);
}

static long face_sites(const hr_ctx *c, int mu) { return c->Vh / c->dims[mu]; }

static void halo_common(HaloArgs &a, const hr_ctx *c, const hr_gauge *links, int parity, int mu)
{
    a.send_up = a.send_dn = nullptr;
    a.recv_prev = a.recv_next = nullptr;
    a.in = nullptr;
    a.out = nullptr;
    a.links = links->data;
    a.parity = parity;
    a.vh = c->Vh;
    a.nface = face_sites(c, mu);
    a.T = c->dims[0]; a.X = c->dims[1]; a.Y = c->dims[2]; a.Zh = c->dims[3] / 2;
    a.beta[0] = a.beta[1] = -0.5;
    a.betaf[0] = a.betaf[1] = -0.5f;
    a.sign_prev = a.sign_next = 1;
}

extern "C" {

size_t hr_face_bytes(const hr_ctx *ctx, hr_prec prec, int mu)
{
    if (!ctx || (prec != HR_F64 && prec != HR_F32) || mu < 0 || mu > 3) return 0;
    return (size_t)face_sites(ctx, mu) * 4 * ctx->d * prec_bytes(prec);
}

size_t hr_halo_bytes(const hr_ctx *ctx, hr_prec prec) { return hr_face_bytes(ctx, prec, 0); }

hr_status hr_dphi_eo_halo_pack(void *send_up, void *send_dn, const void *in, const hr_gauge *links, int parity, void *stream)
{
    return hr_dphi_eo_face_pack(0, send_up, send_dn, in, links, parity, stream);
}

static hr_status check_mu(const char *who, const hr_gauge *links, int mu)
{
    if (mu < 0 || mu > 3) { set_error("%s: direction %d", who, mu); return HR_EINVAL; }
    if (mu == 3 && (links->ctx->dims[2] & 1)) { set_error("%s: a split in z needs an even Y", who); return HR_EINVAL; }
    return HR_OK;
}

hr_status hr_dphi_eo_face_pack(int mu, void *send_up, void *send_dn, const void *in, const hr_gauge *links, int parity, void *stream)
{
    hr_status rc = check_links("hr_dphi_eo_halo_pack", links, parity);
    if (rc != HR_OK) return rc;
    rc = check_mu("hr_dphi_eo_face_pack", links, mu);
    if (rc != HR_OK) return rc;
    if (!send_up || !send_dn || !in) { set_error("hr_dphi_eo_halo_pack: NULL buffer"); return HR_EINVAL; }
    if (!aligned16(send_up) || !aligned16(send_dn) || !aligned16(in) || send_up == send_dn) {
        set_error("hr_dphi_eo_halo_pack: buffers must be distinct and 16-byte aligned");
        return HR_EINVAL;
    }
    HaloArgs a;
    halo_common(a, links->ctx, links, parity, mu);
    a.send_up = send_up;
    a.send_dn = send_dn;
    a.in = in;
    return launch_halo(links->ctx, links->prec, true, mu, a, (cudaStream_t)stream, link_src(links));
}

hr_status hr_dphi_eo_faces_pack(int split_mask, void *const send_up[4], void *const send_dn[4], const void *in, const hr_gauge *links,
                                int parity, void *stream)
{
    hr_status rc = check_links("hr_dphi_eo_faces_pack", links, parity);
    if (rc != HR_OK) return rc;
    if (split_mask <= 0 || split_mask > 15 || !send_up || !send_dn || !in || !aligned16(in)) {
        set_error("hr_dphi_eo_faces_pack: bad argument (split_mask 1..15, non-NULL buffers)");
        return HR_EINVAL;
    }
    HaloArgs a[4];
    int mus[4], n = 0;
    for (int mu = 0; mu < 4; ++mu) {
        if (!(split_mask & (1 << mu))) continue;
        rc = check_mu("hr_dphi_eo_faces_pack", links, mu);
        if (rc != HR_OK) return rc;
        if (!send_up[mu] || !send_dn[mu] || !aligned16(send_up[mu]) || !aligned16(send_dn[mu]) || send_up[mu] == send_dn[mu]) {
            set_error("hr_dphi_eo_faces_pack: buffers of direction %d must be distinct, non-NULL and 16-byte aligned", mu);
            return HR_EINVAL;
        }
        halo_common(a[n], links->ctx, links, parity, mu);
        a[n].send_up = send_up[mu];
        a[n].send_dn = send_dn[mu];
        a[n].in = in;
        mus[n++] = mu;
    }
    return launch_halo_multi(links->ctx, links->prec, true, a, mus, n, (cudaStream_t)stream, link_src(links));
}

hr_status hr_dphi_eo_interior(void *out, const void *in, const hr_gauge *links, int parity, void *stream)
{
    return hr_dphi_eo_interior_mask(out, in, links, parity, 1, stream);
}

hr_status hr_dphi_eo_interior_mask(void *out, const void *in, const hr_gauge *links, int parity, int split_mask, void *stream)
{
    hr_status rc = check_links("hr_dphi_eo_interior", links, parity);
    if (rc != HR_OK) return rc;
    if (split_mask < 0 || split_mask > 15) { set_error("hr_dphi_eo_interior_mask: split_mask=%d", split_mask); return HR_EINVAL; }
    if (!out || !in || out == in || !aligned16(out) || !aligned16(in)) { set_error("hr_dphi_eo_interior: bad buffers"); return HR_EINVAL; }
    const hr_ctx *c = links->ctx;
    DphiArgs a;
    const double zero[2] = { 0.0, 0.0 }, mhalf[2] = { -0.5, -0.5 };
    dphi_args(a, c, out, in, nullptr, links, parity, zero, mhalf);
    // a hop across the boundary of a split direction contributes nothing here: hr_dphi_eo_face_apply adds it
    for (int mu = 0; mu < 4; ++mu)
        if (split_mask & (1 << mu)) a.bc[mu] = 0;
    return launch_dphi(c, links->prec, a, (cudaStream_t)stream, link_src(links));
}

hr_status hr_dphi_eo_halo_apply(void *out, const void *recv_prev, const void *recv_next, const hr_gauge *links, int parity,
                                int first_rank, int last_rank, void *stream)
{
    return hr_dphi_eo_face_apply(0, out, recv_prev, recv_next, links, parity, first_rank, last_rank, stream);
}

hr_status hr_dphi_eo_face_apply(int mu, void *out, const void *recv_prev, const void *recv_next, const hr_gauge *links, int parity,
                                int first_rank, int last_rank, void *stream)
{
    hr_status rc = check_links("hr_dphi_eo_halo_apply", links, parity);
    if (rc != HR_OK) return rc;
    rc = check_mu("hr_dphi_eo_face_apply", links, mu);
    if (rc != HR_OK) return rc;
    if (!out || !recv_prev || !recv_next) { set_error("hr_dphi_eo_halo_apply: NULL buffer"); return HR_EINVAL; }
    if (!aligned16(out) || !aligned16(recv_prev) || !aligned16(recv_next)) {
        set_error("hr_dphi_eo_halo_apply: buffers must be 16-byte aligned");
        return HR_EINVAL;
    }
    const hr_ctx *c = links->ctx;
    HaloArgs a;
    halo_common(a, c, links, parity, mu);
    a.out = out;
    a.recv_prev = recv_prev;
    a.recv_next = recv_next;
    a.sign_prev = first_rank ? c->bc[mu] : 1; // the global seam lies below the first rank's first slice ...
    a.sign_next = last_rank ? c->bc[mu] : 1;  // ... and above the last rank's last slice (reading C9)
    return launch_halo(c, links->prec, false, mu, a, (cudaStream_t)stream, link_src(links));
}

hr_status hr_dphi_eo_faces_apply(int split_mask, void *out, const void *const recv_prev[4], const void *const recv_next[4],
                                 const hr_gauge *links, int parity, int first_mask, int last_mask, void *stream)
{
    hr_status rc = check_links("hr_dphi_eo_faces_apply", links, parity);
    if (rc != HR_OK) return rc;
    if (split_mask <= 0 || split_mask > 15 || !out || !recv_prev || !recv_next || !aligned16(out)) {
        set_error("hr_dphi_eo_faces_apply: bad argument (split_mask 1..15, non-NULL buffers)");
        return HR_EINVAL;
    }
    const hr_ctx *c = links->ctx;
    HaloArgs a[4];
    int mus[4], n = 0;
    for (int mu = 0; mu < 4; ++mu) {
        if (!(split_mask & (1 << mu))) continue;
        rc = check_mu("hr_dphi_eo_faces_apply", links, mu);
        if (rc != HR_OK) return rc;
        if (!recv_prev[mu] || !recv_next[mu] || !aligned16(recv_prev[mu]) || !aligned16(recv_next[mu])) {
            set_error("hr_dphi_eo_faces_apply: buffers of direction %d must be non-NULL and 16-byte aligned", mu);
            return HR_EINVAL;
        }
        halo_common(a[n], c, links, parity, mu);
        a[n].out = out;
        a[n].recv_prev = recv_prev[mu];
        a[n].recv_next = recv_next[mu];
        a[n].sign_prev = (first_mask & (1 << mu)) ? c->bc[mu] : 1;
        a[n].sign_next = (last_mask & (1 << mu)) ? c->bc[mu] : 1;
        mus[n++] = mu;
    }
    // one split direction: the per-direction kernel (compile-time direction) is 2 us faster and bitwise the same
    if (n == 1) return launch_halo(c, links->prec, false, mus[0], a[0], (cudaStream_t)stream, link_src(links));
    return launch_halo_multi(c, links->prec, false, a, mus, n, (cudaStream_t)stream, link_src(links));
}

// ---- face buffers in peer-accessible memory ---------------------------------------------------------------------
// One cudaMalloc allocation of 6 face messages: [send_up | send_dn | recv_prev[0] | recv_next[0] | recv_prev[1] |
// recv_next[1]] (the receive buffers are double-buffered by call parity, see halo.py).  A plain cudaMalloc base pointer
// is what cudaIpcGetMemHandle wants; torch's caching allocator hands out sub-blocks.
hr_status hr_halo_buffers_alloc(const hr_ctx *ctx, hr_prec prec, void **base) { return hr_face_buffers_alloc(ctx, prec, 0, base); }

hr_status hr_face_buffers_alloc(const hr_ctx *ctx, hr_prec prec, int mu, void **base)
{
    if (!ctx || !base || (prec != HR_F64 && prec != HR_F32) || mu < 0 || mu > 3) { set_error("hr_face_buffers_alloc: bad argument"); return HR_EINVAL; }
    *base = nullptr;
    hr_status rc = use_device(ctx);
    if (rc != HR_OK) return rc;
    cudaError_t e = cudaMalloc(base, 6 * hr_face_bytes(ctx, prec, mu));
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail("hr_face_buffers_alloc: cudaMalloc", e); }
    return HR_OK;
}

void hr_halo_buffers_free(const hr_ctx *ctx, void *base)
{
    if (!ctx || !base) return;
    if (cudaSetDevice(ctx->device) == cudaSuccess) cudaFree(base);
    cudaGetLastError();
}

hr_status hr_ipc_export(const hr_ctx *ctx, const void *base, unsigned char handle[64])
{
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "cudaIpcMemHandle_t is 64 bytes");
    if (!ctx || !base || !handle) { set_error("hr_ipc_export: NULL argument"); return HR_EINVAL; }
    hr_status rc = use_device(ctx);
    if (rc != HR_OK) return rc;
    cudaIpcMemHandle_t h;
    cudaError_t e = cudaIpcGetMemHandle(&h, const_cast<void *>(base));
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail("hr_ipc_export: cudaIpcGetMemHandle", e); }
    memcpy(handle, &h, 64);
    return HR_OK;
}

hr_status hr_ipc_open(const hr_ctx *ctx, const unsigned char handle[64], void **peer_base)
{
    if (!ctx || !handle || !peer_base) { set_error("hr_ipc_open: NULL argument"); return HR_EINVAL; }
    *peer_base = nullptr;
    hr_status rc = use_device(ctx);
    if (rc != HR_OK) return rc;
    cudaIpcMemHandle_t h;
    memcpy(&h, handle, 64);
    cudaError_t e = cudaIpcOpenMemHandle(peer_base, h, cudaIpcMemLazyEnablePeerAccess);
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail("hr_ipc_open: cudaIpcOpenMemHandle", e); }
    return HR_OK;
}

hr_status hr_ipc_close(const hr_ctx *ctx, void *peer_base)
{
    if (!ctx || !peer_base) { set_error("hr_ipc_close: NULL argument"); return HR_EINVAL; }
    hr_status rc = use_device(ctx);
    if (rc != HR_OK) return rc;
    cudaError_t e = cudaIpcCloseMemHandle(peer_base);
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail("hr_ipc_close: cudaIpcCloseMemHandle", e); }
    return HR_OK;
}

} // extern "C"
