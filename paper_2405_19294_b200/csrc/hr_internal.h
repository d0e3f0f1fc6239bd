// hr_internal.h -- private structures and device helpers of libhr (sm_100a).
//
// INTERNAL DEVICE LAYOUT.  A per-site record of NREAL reals
// (spinor: 8*d_R; complex link: 2*d^2; real adjoint link: d^2) is cut into 16-byte vectors; vector v
// of all V/2 sites of one parity is one contiguous "plane":
//     address(v, s) = base + (v * Vh + s) * 16          v < NV = NREAL*sizeof(Real)/16
//     tail (NREAL*sizeof(Real) % 16 = 4 or 8 bytes):   base + NV*16*Vh + s*tail_bytes
// s = half index = ((t*X + x)*Y + y)*(Z/2) + z/2 of the site inside its parity.  A warp that walks
// consecutive s therefore issues fully coalesced 128-bit loads (512 contiguous bytes per request).
// Gauge fields hold 8 such record fields, [parity of the link's base site][mu].
// This replaces the paper's per-real strided layout (Fig. 1), which would need four
// (fp32) or two (fp64) times as many load instructions for the same bytes.
#pragma once

#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/hr.h"

struct hr_ctx {
    int dims[4];
    int bc[4];
    int N;
    int rep;
    int d;          // d_R
    int real_links; // adjoint
    int device;
    long V, Vh;
    int variant;    // -1 = default table
    int block;      // 0 = default
    int xblock;     // 0 = default (from the L2 working-set rule), else a divisor of X
    int cg_graph;   // 1 (default): the CG replays one captured iteration as a CUDA graph; 0: plain launches
    int bulk_rows, bulk_stages, bulk_ctas; // bulk kernel (variant 7): rows per tile / ring depth / CTAs per SM; 0 = default
    int bulk_strip; // bulkx kernel (variants 9, 10): tiles per strip; 0 = default
    // host-path workspace (hr_dphi_eo_host)
    void *ws_in, *ws_out, *ws_stage;
    size_t ws_spinor_bytes, ws_stage_bytes;
    int ws_prec;
    // staging of host canonical arrays (hr_gauge_import / export, hr_spinor_import / export, hr_dphi_eo_host): two device
    // buffers and a copy stream, created on first use and kept, so that the copy of chunk k+1 overlaps the (un)packing of chunk k
    void *stage[2];
    size_t stage_bytes;
    cudaStream_t copy_stream;
    cudaEvent_t ev_copied[2], ev_used[2];
    // hr_dphi_eo_host's pipeline: a second copy stream (device -> host) and its events (created with the staging buffers)
    cudaStream_t copy_stream2;
    cudaEvent_t ev_out_ready[2], ev_out_copied[2];
    // device-resident state of hr_qmr_dhat (QmrState + history), created on first use, grown with maxiter
    void *qmr_state;
    size_t qmr_state_bytes;
    // reduction scratch (hr_spinor_dot / norm2, fused Dphi reductions, CG): per-CTA partial sums, the
    // self-resetting ticket counter and a small result area; created on first use, one stream at a time
    void *red_scratch;
    size_t red_scratch_bytes;
};

struct hr_gauge {
    const hr_ctx *ctx;
    int represented;
    hr_prec prec;
    void *data;
    int owns;
    size_t bytes;
    int nreal; // reals per link, internal record (link_nreal)
};

namespace hr {

void set_error(const char *fmt, ...);
void count_launch(int n = 1);
hr_status cuda_fail(const char *what, cudaError_t e);
hr_status use_device(const hr_ctx *c);
hr_status pointer_on_device(const void *p, bool *dev);
struct DphiArgs;
void dphi_args(DphiArgs &a, const hr_ctx *c, void *out, const void *in, const void *self, const hr_gauge *links,
               int parity, const double alpha[2], const double beta[2]);

static inline size_t prec_bytes(hr_prec p) { return p == HR_F64 ? 8 : 4; }
// link-field kinds (hr_gauge::represented): 0 fundamental N x N, 1 represented d_R x d_R, 2 fundamental stored as its
// first N-1 rows (the last row of an SU(N) matrix is fixed by the others; N = 2, 3)
// Row stride of a represented link in the INTERNAL layout.  Real links of an odd d_R > 8 (SU(4) adjoint: 15 x 15) are kept
// with rows of d_R + 1 reals, the last one zero: a row, and a group of 2 (fp64) / 4 (fp32) columns of a row, is then a whole
// number of 16-byte vectors, which is what lets the colour-parallel kernel read U and U^T with vector loads
// (dphi_cp_kernel.cuh).  +6.7 % link bytes; the canonical (import / export) record stays d_R x d_R.  LinkGeom::LD is the
// device-side twin.
static inline int link_ld(const hr_ctx *c) { return (c->real_links && (c->d & 1) && c->d > 8) ? c->d + 1 : c->d; }
// reals per link of the canonical record
static inline int link_nreal_canon(const hr_ctx *c, int represented)
{
    if (represented == 2) return 2 * c->N * (c->N - 1);
    if (!represented) return 2 * c->N * c->N;
    return c->real_links ? c->d * c->d : 2 * c->d * c->d;
}
// reals per link of the internal record
static inline int link_nreal(const hr_ctx *c, int represented)
{
    if (represented == 1 && c->real_links) return c->d * link_ld(c);
    return link_nreal_canon(c, represented);
}

// ---- launch entry points implemented in the kernel translation units ----------------------------
struct DphiArgs {
    void *out;
    const void *in;
    const void *self;  // psi on the output parity, for the (4+m0) term; nullptr for plain Dphi
    const void *links; // represented field, internal layout
    int T, X, Y, Zh;
    int Xb;     // x-block of the thread order (divides X; X = storage order), see dphi_kernel.cuh
    int parity;
    int bc[4];
    long vh;
    // epilogue: out_alpha = alpha[alpha>>1] * self_alpha + beta[alpha>>1] * (sum over the 8 hops)_alpha;
    // index 0 = spin components 0,1, index 1 = components 2,3 (gamma5 = diag(1,1,-1,-1) is a sign
    // pattern on these).  Without self (plain Dphi) the kernel uses beta = -1/2 as a compile-time constant.
    double alpha[2], beta[2];
    float alphaf[2], betaf[2]; // the same, rounded once on the host: constant-bank operands of the fp32 kernels
    // fused reduction of the epilogue (RED): result[0] = sum |out|^2, result[1..2] = <self, out>
    double *red_partial;   // [gridDim.x][3]
    unsigned *red_ticket;  // zero before the launch; the last CTA resets it
    double *red_result;    // [3], device
    const int *skip;       // if non-null and *skip != 0 the launch does nothing (converged CG)
    // fused site-diagonal matrix (clover.cu layout: two packed Hermitian 2 d_R x 2 d_R blocks per site, output parity):
    // site_mode 1: out = alpha self + beta hops + M self;  2: out = M (beta hops);  0: none.  One-thread-per-site kernels.
    const void *site_mat;
    int site_mode;
    // output sites of this launch: the time slices [t0, t0 + Tl) -- the whole lattice (0, T) except for the chunks of
    // hr_dphi_eo_host's copy / compute pipeline; nsite = Tl X Y Zh.  One-thread-per-site kernels only (launch_dphi checks).
    int t0, Tl;
    long nsite;
};

// device-resident state of the CG (cg.cu); the host only reads it
struct CgState {
    double bb;        // |rhs|^2
    double tol2;      // tol^2
    double pap;       // <p, A p> of the current iteration  (= |Q p|^2, written by the fused Dphi reduction)
    double pap_pad[2];
    int iter;         // completed iterations k
    int maxiter;
    int done;         // set by the r-update when rr_k <= tol^2 bb or k == maxiter: later Dphi / r-updates are no-ops
    int frozen;       // set by the first skipped r-update: later x/p-updates are no-ops (the x/p-update of the
                      // iteration that detected convergence still runs)
    // rr[k] = |r_k|^2, k = 0..maxiter, follows this header
};

// launch tuning handed from the context to the kernel launchers
struct LaunchTune {
    int block;                              // CTA size of the site / pair kernels; 0 = default
    int bulk_rows, bulk_stages, bulk_ctas;  // bulk kernel (dphi_bulk_kernel.cuh); 0 = default
    int bulk_strip;                         // bulkx kernel (dphi_bulkx_kernel.cuh); 0 = default
};
static const size_t kMaxDynSmem = 227 * 1024;

// device-resident state of the gamma5-QMR (linalg.cu kernels, hr_qmr_dhat): the Lanczos scalars and Givens rotations never
// leave the device; the host enqueues batches of iterations and reads this header once per batch
struct QmrState {
    double c1, s1, c2, s2, eta, rho, delta, delta_prev, bnorm, tol;
    double alpha, beta;                      // of the current iteration: qmr_scal_a -> Lanczos kernel
    double izeta, eps, theta, ceta, irho;    // qmr_scal_b -> update kernel
    double red[8];                           // [0..1] |vt_up|^2, |vt_lo|^2 (Lanczos kernel); [4..6] fused Dphi reduction: [5] = (v, Dhat v)_J
    int k, maxiter;
    int stop;        // 0 running; 1 |eta_k| <= tol |b|: the host checks the TRUE residual; 2 breakdown (delta = 0 or zeta = 0);
                     // 3 Krylov space exhausted (rho_{k+1} = 0); 4 k = maxiter.  Non-zero: every later kernel is a no-op
    int do_update;   // the update kernel of the current iteration runs (0 for skipped iterations and after zeta = 0)
    // hist[k] = |eta_k| / |b|, k = 0..maxiter, follows
};

// number of CTAs the reduction scratch provides partial-sum slots for
static const unsigned kRedMaxBlocks = 1u << 20;
struct RedScratch {
    double *partial;
    unsigned *ticket;
    double *result;
};
hr_status get_red_scratch(hr_ctx *c, RedScratch *r, cudaStream_t st);

// returns HR_OK / HR_EUNSUPPORTED / HR_ECUDA
// link_src: what a.links holds -- 0 the represented field, 1 the FUNDAMENTAL field (representation applied on the fly,
// NEXT-3), 2 the fundamental field stored as N-1 rows (last row and representation rebuilt in the kernel)
hr_status launch_dphi(const hr_ctx *c, hr_prec prec, const DphiArgs &a, cudaStream_t st, int link_src = 0);
int dphi_link_kind(const hr_ctx *c, int link_src); // -1: no such kernel
static inline int link_src(const hr_gauge *g) { return g->represented == 1 ? 0 : g->represented == 0 ? 1 : 2; }
hr_status launch_compress(const hr_ctx *c, hr_prec prec, void *rows, const void *fund, cudaStream_t st);
bool dphi_site_fusable(const hr_ctx *c, hr_prec prec, int link_src);
const char *dphi_variant_name(const hr_ctx *c, hr_prec prec);
bool dphi_variant_valid(const hr_ctx *c, int variant);

// slab decomposition along t (halo_kernel.cuh)
struct HaloArgs {
    void *send_up;         // to the next rank:  chi = U_0^dagger P+ psi of my last slice     (pack)
    void *send_dn;         // to the previous rank: h = P- psi of my first slice                (pack)
    const void *recv_prev; // the previous rank's send_up                                       (apply)
    const void *recv_next; // the next rank's send_dn                                           (apply)
    const void *in;        // pack: parity-(1-p) half field
    void *out;             // apply: parity-p half field, already holding the interior result
    const void *links;
    int parity;            // p, parity of the OUTPUT sites of the Dphi_eo being assembled
    long vh, nface;        // V_local/2; face sites of the direction (V_local/2 / L_mu)
    int T, X, Y, Zh;       // local extents
    double beta[2];        // coefficient of the hop sum in the interior launch (-1/2 for plain Dphi)
    float betaf[2];
    int sign_prev, sign_next; // seam signs of the two faces (+-1)
};
hr_status launch_halo(const hr_ctx *c, hr_prec prec, bool pack, int mu, const HaloArgs &a, cudaStream_t st, int link_src);
hr_status launch_halo_multi(const hr_ctx *c, hr_prec prec, bool pack, const HaloArgs *a, const int *mu, int ndir, cudaStream_t st, int link_src);

// clover term (clover.cu): record of 8 d_R^2 reals per site, [parity] fields
size_t clover_nreal(const hr_ctx *c);
hr_status launch_clover_build(const hr_ctx *c, hr_prec prec, void *clover, const void *links, double csw, cudaStream_t st);
hr_status launch_clover_exp(const hr_ctx *c, hr_prec prec, void *clover, double m, cudaStream_t st);
hr_status launch_clover_apply(const hr_ctx *c, hr_prec prec, void *out, const void *in, const void *clover_parity, cudaStream_t st,
                              int mode = 1);
hr_status launch_clover_finalize(const hr_ctx *c, hr_prec prec, void *clover, void *inverse, double m, cudaStream_t st);

hr_status launch_represent(const hr_ctx *c, hr_prec in_prec, const void *fund, hr_prec out_prec, void *repr,
                           cudaStream_t st);

// spinor linear algebra on internal-layout half fields (linalg.cu).  nvec = 16-byte vectors per field.
//   out = ca * G(x) + cb * y   (G = gamma5 if g5 else identity; y may be null; out may alias x or y)
hr_status launch_lincomb(const hr_ctx *c, hr_prec prec, void *out, const double ca[2], int g5, const void *x,
                         const double cb[2], const void *y, cudaStream_t st);
// half field fp64 -> fp32 (dst = (float)(scale * src)) when down, else fp64 accumulate dst += scale * (double) src
hr_status launch_cvt(const hr_ctx *c, bool down, void *dst, const void *src, double scale, cudaStream_t st);
//   result[0..1] = <x, y> (result[0] = |x|^2 when x == y), device pointer
hr_status launch_dot(const hr_ctx *c, hr_prec prec, const void *x, const void *y, const RedScratch &rs,
                     double *result_dev, cudaStream_t st);
// one QMR iteration's vector work and scalar recurrences on the device-resident QmrState
hr_status launch_qmr_init(QmrState *qs, double bnorm, double delta0, double tol, int maxiter, cudaStream_t st);
hr_status launch_qmr_scal_a(QmrState *qs, cudaStream_t st);
hr_status launch_qmr_lanczos(const hr_ctx *c, hr_prec prec, void *w, const void *v, const void *vp, QmrState *qs, const RedScratch &rs,
                             cudaStream_t st);
hr_status launch_qmr_scal_b(QmrState *qs, cudaStream_t st);
hr_status launch_qmr_update(const hr_ctx *c, hr_prec prec, void *p2, const void *p1, const void *v, void *x, void *vp, const void *w,
                            const QmrState *qs, cudaStream_t st);
hr_status launch_qmr_resume(QmrState *qs, cudaStream_t st);
hr_status launch_dot_range(const hr_ctx *c, hr_prec prec, const void *x, const void *y, size_t first, size_t nvec,
                           const RedScratch &rs, double *result_dev, cudaStream_t st);
// CG building blocks on the device-resident CgState (cg.cu)
hr_status launch_cg_init(const hr_ctx *c, hr_prec prec, CgState *cs, double tol, int maxiter, void *x, void *p,
                         const void *r, const RedScratch &rs, cudaStream_t st);
hr_status launch_cg_update_r(const hr_ctx *c, hr_prec prec, CgState *cs, void *r, const void *Ap,
                             const RedScratch &rs, cudaStream_t st);
hr_status launch_cg_update_xp(const hr_ctx *c, hr_prec prec, const CgState *cs, void *x, void *p, const void *r,
                              cudaStream_t st);

// BiCGstab building blocks on a device-resident state (bicgstab.cu); the state struct is private to that file
size_t bicgstab_state_bytes(int maxiter);
size_t bicgstab_header_bytes();
double *bicgstab_rhat_v(void *state);
double *bicgstab_tt_st(void *state);
const int *bicgstab_done(void *state);
void bicgstab_unpack(const void *host_copy, int *iter, int *done, double *bb);
hr_status launch_bi_init(const hr_ctx *c, hr_prec prec, void *state, double tol, int maxiter, void *x, void *r, void *rhat,
                         void *p, void *v, const void *b, const RedScratch &rs, cudaStream_t st);
hr_status launch_bi_update_p(const hr_ctx *c, hr_prec prec, const void *state, void *p, const void *r, const void *v, cudaStream_t st);
hr_status launch_bi_update_s(const hr_ctx *c, hr_prec prec, void *state, void *s, const void *r, const void *v, cudaStream_t st);
hr_status launch_bi_update_xr(const hr_ctx *c, hr_prec prec, void *state, void *x, void *r, const void *p, const void *s,
                              const void *t, const void *rhat, const RedScratch &rs, cudaStream_t st);

// pack / unpack: canonical AoS (device pointer) <-> internal planes
hr_status launch_pack_spinor(const hr_ctx *c, void *dst, hr_prec prec, const void *canon_dev, hr_prec cprec,
                             long first_site, long nsites, cudaStream_t st);
hr_status launch_unpack_spinor(const hr_ctx *c, const void *src, hr_prec prec, void *canon_dev, hr_prec cprec,
                               long first_site, long nsites, cudaStream_t st);
// nreal: reals of the internal record; ld / dcol: internal row stride and canonical row length when they differ (link_ld),
// 0 / 0 otherwise
hr_status launch_pack_gauge(const hr_ctx *c, int nreal, int ld, int dcol, void *dst, hr_prec prec, const void *canon_dev,
                            hr_prec cprec, long first_site, long nsites, cudaStream_t st);
hr_status launch_unpack_gauge(const hr_ctx *c, int nreal, int ld, int dcol, const void *src, hr_prec prec, void *canon_dev,
                              hr_prec cprec, long first_site, long nsites, cudaStream_t st);

} // namespace hr

// =================================================================================================
// device-side helpers
// =================================================================================================
#ifdef __CUDACC__
namespace hr {

template <typename Real> struct VecOf;
template <> struct VecOf<double> { static constexpr int RPV = 2; };
template <> struct VecOf<float> { static constexpr int RPV = 4; };

// record geometry
template <typename Real, int NREAL> struct Rec {
    static constexpr int RPV = 16 / (int)sizeof(Real);
    static constexpr int NV = NREAL / RPV;
    static constexpr int TAIL = NREAL - NV * RPV; // reals in the tail plane
    static constexpr int BYTES = NREAL * (int)sizeof(Real);
};

// cache-hint flavours of a 16-byte global load (all read-only path, .nc)
enum : int {
    LD_DEFAULT = 0,   // ld.global.nc               : allocate in L1 and L2 (neighbour spinors: re-used)
    LD_STREAM = 1,    // + L1::no_allocate          : touched once per call (links)
    LD_STREAM_EF = 2, // + L2 evict_first policy    : links must not push spinors out of L2
    LD_KEEP = 3       // default L1 + L2 evict_last : neighbour spinors at volumes whose time-slice exceeds L2
};

__device__ __forceinline__ uint64_t make_policy_evict_first()
{
    uint64_t p;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t make_policy_evict_last()
{
    uint64_t p;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}

template <int HINT> __device__ __forceinline__ void ld16(double &a, double &b, const void *p, uint64_t pol)
{
    if constexpr (HINT == LD_DEFAULT)
        asm("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(a), "=d"(b) : "l"(p));
    else if constexpr (HINT == LD_STREAM)
        asm("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(a), "=d"(b) : "l"(p));
    else if constexpr (HINT == LD_STREAM_EF)
        asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;"
            : "=d"(a), "=d"(b) : "l"(p), "l"(pol));
    else
        asm("ld.global.nc.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(a), "=d"(b) : "l"(p), "l"(pol));
}
template <int HINT>
__device__ __forceinline__ void ld16(float &a, float &b, float &c, float &d, const void *p, uint64_t pol)
{
    if constexpr (HINT == LD_DEFAULT)
        asm("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(a), "=f"(b), "=f"(c), "=f"(d) : "l"(p));
    else if constexpr (HINT == LD_STREAM)
        asm("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
            : "=f"(a), "=f"(b), "=f"(c), "=f"(d) : "l"(p));
    else if constexpr (HINT == LD_STREAM_EF)
        asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
            : "=f"(a), "=f"(b), "=f"(c), "=f"(d) : "l"(p), "l"(pol));
    else
        asm("ld.global.nc.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
            : "=f"(a), "=f"(b), "=f"(c), "=f"(d) : "l"(p), "l"(pol));
}
template <int HINT> __device__ __forceinline__ void ld8(double &a, const void *p, uint64_t pol)
{
    if constexpr (HINT == LD_DEFAULT)
        asm("ld.global.nc.f64 %0, [%1];" : "=d"(a) : "l"(p));
    else if constexpr (HINT == LD_STREAM)
        asm("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(a) : "l"(p));
    else if constexpr (HINT == LD_STREAM_EF)
        asm("ld.global.nc.L1::no_allocate.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(a) : "l"(p), "l"(pol));
    else
        asm("ld.global.nc.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(a) : "l"(p), "l"(pol));
}
template <int HINT> __device__ __forceinline__ void ld8(float &a, float &b, const void *p, uint64_t pol)
{
    if constexpr (HINT == LD_DEFAULT)
        asm("ld.global.nc.v2.f32 {%0,%1}, [%2];" : "=f"(a), "=f"(b) : "l"(p));
    else if constexpr (HINT == LD_STREAM)
        asm("ld.global.nc.L1::no_allocate.v2.f32 {%0,%1}, [%2];" : "=f"(a), "=f"(b) : "l"(p));
    else if constexpr (HINT == LD_STREAM_EF)
        asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;"
            : "=f"(a), "=f"(b) : "l"(p), "l"(pol));
    else
        asm("ld.global.nc.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;" : "=f"(a), "=f"(b) : "l"(p), "l"(pol));
}
template <int HINT> __device__ __forceinline__ void ld4(float &a, const void *p, uint64_t pol)
{
    if constexpr (HINT == LD_DEFAULT)
        asm("ld.global.nc.f32 %0, [%1];" : "=f"(a) : "l"(p));
    else if constexpr (HINT == LD_STREAM)
        asm("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(a) : "l"(p));
    else if constexpr (HINT == LD_STREAM_EF)
        asm("ld.global.nc.L1::no_allocate.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(a) : "l"(p), "l"(pol));
    else
        asm("ld.global.nc.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(a) : "l"(p), "l"(pol));
}

// NVEC consecutive planes starting at `p` (= address of the first plane's element for this site)
template <int HINT, int NVEC>
__device__ __forceinline__ void load_planes(double *dst, const char *p, size_t plane_bytes, uint64_t pol)
{
#pragma unroll
    for (int v = 0; v < NVEC; ++v) ld16<HINT>(dst[2 * v], dst[2 * v + 1], p + v * plane_bytes, pol);
}
template <int HINT, int NVEC>
__device__ __forceinline__ void load_planes(float *dst, const char *p, size_t plane_bytes, uint64_t pol)
{
#pragma unroll
    for (int v = 0; v < NVEC; ++v)
        ld16<HINT>(dst[4 * v], dst[4 * v + 1], dst[4 * v + 2], dst[4 * v + 3], p + v * plane_bytes, pol);
}

// whole record of NREAL reals of site s from the record field at `base`
template <int HINT, int NREAL>
__device__ __forceinline__ void load_record(double (&dst)[NREAL], const char *base, size_t vh, size_t s, uint64_t pol)
{
    using R = Rec<double, NREAL>;
    load_planes<HINT, R::NV>(dst, base + s * 16, vh * 16, pol);
    if constexpr (R::TAIL == 1) ld8<HINT>(dst[NREAL - 1], base + (size_t)R::NV * 16 * vh + s * 8, pol);
}
template <int HINT, int NREAL>
__device__ __forceinline__ void load_record(float (&dst)[NREAL], const char *base, size_t vh, size_t s, uint64_t pol)
{
    using R = Rec<float, NREAL>;
    load_planes<HINT, R::NV>(dst, base + s * 16, vh * 16, pol);
    const char *t = base + (size_t)R::NV * 16 * vh;
    if constexpr (R::TAIL == 1) ld4<HINT>(dst[NREAL - 1], t + s * 4, pol);
    if constexpr (R::TAIL == 2) ld8<HINT>(dst[NREAL - 2], dst[NREAL - 1], t + s * 8, pol);
    if constexpr (R::TAIL == 3) {
        ld4<HINT>(dst[NREAL - 3], t + s * 12, pol);
        ld4<HINT>(dst[NREAL - 2], t + s * 12 + 4, pol);
        ld4<HINT>(dst[NREAL - 1], t + s * 12 + 8, pol);
    }
}

// stores (output spinor: written once, never re-read by this kernel -> streaming)
enum : int { ST_DEFAULT = 0, ST_STREAM = 1 };
template <int HINT> __device__ __forceinline__ void st16(void *p, double a, double b)
{
    if constexpr (HINT == ST_DEFAULT)
        asm volatile("st.global.v2.f64 [%0], {%1,%2};" ::"l"(p), "d"(a), "d"(b) : "memory");
    else
        asm volatile("st.global.cs.v2.f64 [%0], {%1,%2};" ::"l"(p), "d"(a), "d"(b) : "memory");
}
template <int HINT> __device__ __forceinline__ void st16(void *p, float a, float b, float c, float d)
{
    if constexpr (HINT == ST_DEFAULT)
        asm volatile("st.global.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
    else
        asm volatile("st.global.cs.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
template <int HINT, int NVEC>
__device__ __forceinline__ void store_planes(char *p, size_t plane_bytes, const double *src)
{
#pragma unroll
    for (int v = 0; v < NVEC; ++v) st16<HINT>(p + v * plane_bytes, src[2 * v], src[2 * v + 1]);
}
template <int HINT, int NVEC>
__device__ __forceinline__ void store_planes(char *p, size_t plane_bytes, const float *src)
{
#pragma unroll
    for (int v = 0; v < NVEC; ++v)
        st16<HINT>(p + v * plane_bytes, src[4 * v], src[4 * v + 1], src[4 * v + 2], src[4 * v + 3]);
}


// whole record of NREAL reals of site s into the record field at `base` (default cache policy)
template <int NREAL>
__device__ __forceinline__ void store_record(char *base, size_t vh, size_t s, const double (&src)[NREAL])
{
    using R = Rec<double, NREAL>;
    store_planes<ST_DEFAULT, R::NV>(base + s * 16, vh * 16, src);
    if constexpr (R::TAIL == 1) *(double *)(base + (size_t)R::NV * 16 * vh + s * 8) = src[NREAL - 1];
}
template <int NREAL>
__device__ __forceinline__ void store_record(char *base, size_t vh, size_t s, const float (&src)[NREAL])
{
    using R = Rec<float, NREAL>;
    store_planes<ST_DEFAULT, R::NV>(base + s * 16, vh * 16, src);
    float *t = (float *)(base + (size_t)R::NV * 16 * vh) + s * R::TAIL;
#pragma unroll
    for (int e = 0; e < R::TAIL; ++e) t[e] = src[R::NV * 4 + e];
}

// ---- one-pass grid reduction (replaces the paper's two-kernel cub scheme) -------------
// Every CTA reduces its threads' NRED fp64 partial sums (shuffle tree, then a fixed-order sum over the
// warps), writes them to partial[blockIdx.x][NRED] and takes a ticket; the CTA that draws the last ticket
// sums the per-CTA partials in an order that depends only on the launch geometry -- the result is
// bitwise reproducible run to run (reading C15) -- and leaves the totals in v[] of its thread 0.
// Returns true on exactly that thread.  atomicInc wraps the ticket back to 0 for the next launch.
template <int NRED>
__device__ __forceinline__ bool grid_reduce(double (&v)[NRED], double *partial, unsigned *ticket)
{
    __shared__ double sm[32][NRED];
    __shared__ bool last;
    const int tid = threadIdx.x + threadIdx.y * blockDim.x;
    const int nthr = blockDim.x * blockDim.y;
    const int lane = tid & 31, warp = tid >> 5, nwarp = (nthr + 31) >> 5;
    auto block_sum = [&]() {
#pragma unroll
        for (int i = 0; i < NRED; ++i)
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], o);
        if (lane == 0)
#pragma unroll
            for (int i = 0; i < NRED; ++i) sm[warp][i] = v[i];
        __syncthreads();
        if (tid == 0)
#pragma unroll
            for (int i = 0; i < NRED; ++i) {
                double t = 0;
                for (int w = 0; w < nwarp; ++w) t += sm[w][i];
                v[i] = t;
            }
    };
    block_sum();
    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < NRED; ++i) partial[(size_t)blockIdx.x * NRED + i] = v[i];
        __threadfence();
        const unsigned t = atomicInc(ticket, gridDim.x - 1);
        last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!last) return false;
    __threadfence();
#pragma unroll
    for (int i = 0; i < NRED; ++i) {
        double t = 0;
        for (unsigned b = tid; b < gridDim.x; b += nthr) t += __ldcg(&partial[(size_t)b * NRED + i]);
        v[i] = t;
    }
    __syncthreads(); // sm is re-used
    block_sum();
    return tid == 0;
}

} // namespace hr
#endif // __CUDACC__
