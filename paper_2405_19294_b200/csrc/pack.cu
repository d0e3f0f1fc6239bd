// pack.cu -- canonical AoS <-> internal 16-byte-plane layout.
// Pure permutation + one precision conversion; set-up path, not part of the timed hot path
// (only hr_dphi_eo_host uses it per call, where PCIe dominates).
#include "hr_internal.h"

namespace hr {

// One thread per (site, 16-byte vector of the internal record).  blockDim = (32 sites, VY vectors):
// the plane writes are coalesced over sites, the canonical reads of a block cover one contiguous
// range of 32 records.
template <typename TC, typename TI, bool PACK, bool GAUGE>
__global__ void pack_kernel(char *internal, TC *canon, int nreal, int ld, int dcol, long first_site, long nsites, long vh, int X,
                            int Y, int Z)
{
    // ld > 0: the internal record has rows of ld reals of which the first dcol are the canonical row (hr_internal.h link_ld)
    const int cn = ld > 0 ? nreal / ld * dcol : nreal;   // reals of the canonical record
    constexpr int RPV = 16 / (int)sizeof(TI);
    const int nv = nreal / RPV, tail = nreal - nv * RPV;
    const int nvt = nv + (tail ? 1 : 0);
    const int nrec = GAUGE ? 4 : 1; // records per site (4 links)
    const long j = (long)blockIdx.x * blockDim.x + threadIdx.x; // site within the chunk
    if (j >= nsites) return;
    const long i = first_site + j; // spinor: half index; gauge: full-lattice index
    long s = i;
    int q = 0;
    if constexpr (GAUGE) {
        long r = i;
        const int z = (int)(r % Z); r /= Z;
        const int y = (int)(r % Y); r /= Y;
        const int x = (int)(r % X);
        const int t = (int)(r / X);
        q = (t + x + y + z) & 1;
        s = i >> 1;
    }
    const size_t rec_bytes = (size_t)nreal * sizeof(TI);
    for (int w = threadIdx.y; w < nrec * nvt; w += blockDim.y) {
        const int mu = w / nvt, v = w % nvt;
        char *field = internal + (size_t)(q * nrec + mu) * rec_bytes * (size_t)vh;
        TC *crec = canon + ((size_t)j * nrec + mu) * cn;
        TI *p;
        int cnt;
        if (v < nv) { p = (TI *)(field + ((size_t)v * vh + s) * 16); cnt = RPV; }
        else        { p = (TI *)(field + (size_t)nv * 16 * vh + (size_t)s * tail * sizeof(TI)); cnt = tail; }
        for (int e = 0; e < cnt; ++e) {
            int ce = v * RPV + e;
            if (ld > 0) {
                const int row = ce / ld, col = ce - row * ld;
                if (col >= dcol) { if constexpr (PACK) p[e] = (TI)0; continue; }
                ce = row * dcol + col;
            }
            if constexpr (PACK) p[e] = (TI)crec[ce];
            else crec[ce] = (TC)p[e];
        }
    }
}

template <bool PACK, bool GAUGE>
static hr_status run(const hr_ctx *c, int nreal, int ld, int dcol, void *internal, hr_prec prec, void *canon, hr_prec cprec,
                     long first_site, long nsites, cudaStream_t st)
{
    if (nsites <= 0) return HR_OK;
    const int rpv = prec == HR_F64 ? 2 : 4;
    const int nvt = (nreal + rpv - 1) / rpv;
    int vy = (GAUGE ? 4 : 1) * nvt;
    if (vy > 16) vy = 16;
    dim3 block(32, vy);
    dim3 grid((unsigned)((nsites + 31) / 32));
    const int X = c->dims[1], Y = c->dims[2], Z = c->dims[3];
#define LAUNCH(TC, TI) pack_kernel<TC, TI, PACK, GAUGE><<<grid, block, 0, st>>>((char *)internal, (TC *)canon, nreal, ld, dcol, first_site, nsites, c->Vh, X, Y, Z)
    if (cprec == HR_F64 && prec == HR_F64) LAUNCH(double, double);
    else if (cprec == HR_F64 && prec == HR_F32) LAUNCH(double, float);
    else if (cprec == HR_F32 && prec == HR_F64) LAUNCH(float, double);
    else LAUNCH(float, float);
#undef LAUNCH
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { set_error("pack kernel launch failed: %s", cudaGetErrorString(e)); return HR_ECUDA; }
    return HR_OK;
}

hr_status launch_pack_spinor(const hr_ctx *c, void *dst, hr_prec prec, const void *canon_dev, hr_prec cprec,
                             long first_site, long nsites, cudaStream_t st)
{ return run<true, false>(c, 8 * c->d, 0, 0, dst, prec, const_cast<void *>(canon_dev), cprec, first_site, nsites, st); }

hr_status launch_unpack_spinor(const hr_ctx *c, const void *src, hr_prec prec, void *canon_dev, hr_prec cprec,
                               long first_site, long nsites, cudaStream_t st)
{ return run<false, false>(c, 8 * c->d, 0, 0, const_cast<void *>(src), prec, canon_dev, cprec, first_site, nsites, st); }

hr_status launch_pack_gauge(const hr_ctx *c, int nreal, int ld, int dcol, void *dst, hr_prec prec, const void *canon_dev,
                            hr_prec cprec, long first_site, long nsites, cudaStream_t st)
{ return run<true, true>(c, nreal, ld, dcol, dst, prec, const_cast<void *>(canon_dev), cprec, first_site, nsites, st); }

hr_status launch_unpack_gauge(const hr_ctx *c, int nreal, int ld, int dcol, const void *src, hr_prec prec, void *canon_dev,
                              hr_prec cprec, long first_site, long nsites, cudaStream_t st)
{ return run<false, true>(c, nreal, ld, dcol, const_cast<void *>(src), prec, canon_dev, cprec, first_site, nsites, st); }

} // namespace hr
