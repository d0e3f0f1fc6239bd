// dphi_launch.cuh -- variant table + launcher for one (Real, D, real-link) combination.
// Each dphi_inst_*.cu includes this and instantiates launch_dphi_t for its combination, so the
// combinations compile in parallel.
#pragma once
#include <type_traits>

#include "dphi_kernel.cuh"
#ifdef HR_BUILD_EXPERIMENTS
// variants that were measured and lost everywhere (DESIGN.md sections 7, 14); kept as evidence, not in the default build
#include "dphi_pf_kernel.cuh"
#include "dphi_cpo_kernel.cuh"
#include "dphi_loop_kernel.cuh"
#endif
#include "dphi_cp_kernel.cuh"
#include "dphi_bulk_kernel.cuh"
#include "dphi_bulkx_kernel.cuh"
#include "halo_kernel.cuh"

namespace hr {

// Kernel variants (hr_ctx_set_tuning "variant"); names are what bench.py / profiles report.
//   0 site      one thread per site, links streamed past L1
//   1 site_ef   + links evict-first in L2, neighbour spinors evict-last (large volumes)
//   2 pair      two threads per site (one per half-spinor component)
//   3 pair_ef   pair + the L2 policies of 1
//   4 site_l1   one thread per site, links through L1 as well (baseline for the cache-policy evidence)
//   5 site_pf   one thread per site, the next hop's operands prefetched with cp.async into a private,
//               double-buffered shared-memory stage (dphi_pf_kernel.cuh)
//   6 colour    one thread per (site, colour row): the large-d_R kernel (dphi_cp_kernel.cuh; represented links)
//   7 bulk      persistent CTAs, operands of every hop staged in shared memory by TMA bulk copies (dphi_bulk_kernel.cuh)
//   8 bulk2     the same with two consumer threads per site (one per half-spinor component)
//   9 bulkx     bulk + the neighbour spinors of a time-slice kept in shared memory along a strip in x and re-used across
//               sites (dphi_bulkx_kernel.cuh); d_R <= 4
//  10 bulkx2    bulkx with two consumer threads per site
//  11 site_loop one thread per site, the four directions as a loop with run-time projectors (dphi_loop_kernel.cuh): a
//               quarter of the code.  Measured 8-16 % SLOWER than `site` on every case (the loop stops ptxas hoisting the
//               next direction's loads above this direction's arithmetic): -DHR_BUILD_EXPERIMENTS only
// d_R > 8 (SU(4) two-index symmetric, adjoint) compiles only 0 (the paper's "unimproved" kernel, for comparison) and 6.
// Variants 4, 5 and the colour-parallel on-the-fly kernel lost every measurement: they are compiled only with
// -DHR_BUILD_EXPERIMENTS; the pair kernels (2, 3) only where they were ever competitive (d_R >= 6).
enum { DPHI_NVARIANTS = 12 };
#ifdef HR_BUILD_EXPERIMENTS
static constexpr bool kExperiments = true;
#else
static constexpr bool kExperiments = false;
#endif

// registers: __launch_bounds__(MAXT, MINB) caps them at 65536 / (MAXT*MINB)
// LIVE in (96, 128] (the fp32 d_R = 3 kernels) at a 128-register cap: ptxas parks the upper halves of two or three
// loop-invariant 64-bit addresses in local memory (2-3 STL at the top of the kernel, 2-3 LDL before the epilogue: 8-28
// bytes per thread, L1-resident).  It does the same at a 168-register cap (checked: -DHR_MINB_128=3 gives "168 registers,
// 8 bytes spill" -- the scheduler hoists loads until the budget is full), so the cap stays where the time is best.
#ifndef HR_OTF32_MINB
#define HR_OTF32_MINB 4
#endif
#ifndef HR_MINB_128
#define HR_MINB_128 4
#endif
template <typename Real, int D, int LK, int KSPLIT> struct Tune {
    static constexpr int LNREAL = LinkGeom<LK, D>::NREAL;
    // live values of a thread, in 32-bit registers (accumulators + one spinor/half + one link)
    static constexpr int W = (int)sizeof(Real) / 4;
    static constexpr int LIVE = W * ((KSPLIT == 1 ? 8 * D : 6 * D) + (KSPLIT == 1 ? 8 * D : 4 * D) + LNREAL) + 40;
    static constexpr int MAXT = 128;
    // measured (profiles/): the fp32 on-the-fly kernels gain 7 % from a 128-register cap (16 warps per SM); the fp64
    // real-link d_R = 3 kernel (LIVE = 154) loses 3 % at a 168-register cap (it spills), hence the 150 threshold
    static constexpr int MINB = ((LK == LK_SYM_OTF || LK == LK_ASYM_OTF) && sizeof(Real) == 4 && KSPLIT == 1) ? HR_OTF32_MINB :
                                (LK == LK_ADJ2_ROWS && sizeof(Real) == 8 && KSPLIT == 1) ? 2 :   // as the real-link kernel it expands to
                                LIVE <= 64 ? 8 : LIVE <= 80 ? 6 : LIVE <= 96 ? 5 : LIVE <= 128 ? HR_MINB_128 : LIVE <= 150 ? 3 : LIVE <= 255 ? 2 : 1;
};

template <typename Real, int D, int LK, int KSPLIT, bool MASS, bool RED, int LHINT, int SHINT, int STHINT, int CLV = 0>
static hr_status launch_one(int block, const DphiArgs &a, cudaStream_t st)
{
    using T = Tune<Real, D, LK, KSPLIT>;
    // default CTA: 64 threads for the one-thread-per-site kernels (same warps per SM, finer tail; measured 1-4 %
    // faster than 128 on every config), 128 for the pair kernels
    if (block <= 0) block = KSPLIT == 1 ? 64 : T::MAXT;
    if (block > T::MAXT || (block % 32) != 0) {
        set_error("block=%d not supported by this variant (multiple of 32, <= %d)", block, T::MAXT);
        return HR_EINVAL;
    }
    const long nthreads = a.nsite * KSPLIT;
    const long grid = (nthreads + block - 1) / block;
    if (RED && (unsigned long)grid > kRedMaxBlocks) {
        set_error("fused Dphi reduction: %ld CTAs exceed the reduction scratch (%u)", grid, kRedMaxBlocks);
        return HR_EUNSUPPORTED;
    }
#if HR_PDL
    {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)grid);
        cfg.blockDim = dim3((unsigned)block);
        cfg.dynamicSmemBytes = 0;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        cudaError_t le = cudaLaunchKernelEx(&cfg, dphi_kernel<Real, D, LK, KSPLIT, MASS, RED, LHINT, SHINT, STHINT, T::MAXT, T::MINB, CLV>, a);
        if (le != cudaSuccess) { set_error("dphi kernel launch failed: %s", cudaGetErrorString(le)); cudaGetLastError(); return HR_ECUDA; }
    }
#else
    dphi_kernel<Real, D, LK, KSPLIT, MASS, RED, LHINT, SHINT, STHINT, T::MAXT, T::MINB, CLV><<<(unsigned)grid, block, 0, st>>>(a);
#endif
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) {
        set_error("dphi kernel launch failed: %s", cudaGetErrorString(e));
        return HR_ECUDA;
    }
    return HR_OK;
}

#ifdef HR_BUILD_EXPERIMENTS
template <typename Real, int D, int LK, bool MASS, bool RED>
static hr_status launch_pf(int block, const DphiArgs &a, cudaStream_t st)
{
    using T = Tune<Real, D, LK, 1>;
    using G = PfGeom<Real, D, LK>;
    if (block <= 0) block = G::smem_bytes(T::MAXT) * 2 <= kMaxDynSmem ? T::MAXT : 64; // at least two CTAs per SM
    if (block > T::MAXT || (block % 32) != 0 || G::smem_bytes(block) > kMaxDynSmem) {
        set_error("site_pf: block=%d needs %zu bytes of shared memory (max %zu)", block, G::smem_bytes(block), kMaxDynSmem);
        return HR_EUNSUPPORTED;
    }
    auto kern = dphi_pf_kernel<Real, D, LK, MASS, RED, T::MAXT, T::MINB>;
    static bool attr_set[64] = {}; // per instantiation and device (the attribute lives in the device's context)
    int dev = 0;
    cudaGetDevice(&dev);
    if (!(dev >= 0 && dev < 64 && attr_set[dev])) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxDynSmem);
        if (e != cudaSuccess) { set_error("site_pf: cudaFuncSetAttribute: %s", cudaGetErrorString(e)); cudaGetLastError(); return HR_ECUDA; }
        if (dev >= 0 && dev < 64) attr_set[dev] = true;
    }
    const long grid = (a.vh + block - 1) / block;
    if (RED && (unsigned long)grid > kRedMaxBlocks) { set_error("fused Dphi reduction: too many CTAs"); return HR_EUNSUPPORTED; }
    kern<<<(unsigned)grid, block, G::smem_bytes(block), st>>>(a);
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { set_error("dphi_pf kernel launch failed: %s", cudaGetErrorString(e)); return HR_ECUDA; }
    return HR_OK;
}
#endif

#ifdef HR_BUILD_EXPERIMENTS
template <typename Real, int D, int LK, bool MASS, bool RED>
static hr_status launch_loop(int block, const DphiArgs &a, cudaStream_t st)
{
    using T = Tune<Real, D, LK, 1>;
    if (block <= 0) block = 64;
    if (block > T::MAXT || (block % 32) != 0) { set_error("block=%d not supported by this variant (multiple of 32, <= %d)", block, T::MAXT); return HR_EINVAL; }
    const long grid = (a.vh + block - 1) / block;
    if (RED && (unsigned long)grid > kRedMaxBlocks) { set_error("fused Dphi reduction: too many CTAs"); return HR_EUNSUPPORTED; }
    dphi_loop_kernel<Real, D, LK, MASS, RED, LD_STREAM, LD_DEFAULT, T::MAXT, T::MINB><<<(unsigned)grid, block, 0, st>>>(a);
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { set_error("dphi loop kernel launch failed: %s", cudaGetErrorString(e)); return HR_ECUDA; }
    return HR_OK;
}
#endif

template <typename Real, int D, int LK, bool MASS, bool RED>
static hr_status launch_variant(int variant, const LaunchTune &lt, const DphiArgs &a, cudaStream_t st)
{
    constexpr int RPV = 16 / (int)sizeof(Real);
    constexpr bool PAIR_OK = (2 * D) % RPV == 0 && (D >= 6 || kExperiments);
    constexpr bool CP_OK = (LK == LK_COMPLEX || LK == LK_REAL);
    const int block = lt.block;
    if constexpr (CP_OK) {
        if (variant == 6) return launch_cp<Real, D, LK, MASS, RED>(a, st);
    }
#ifdef HR_BUILD_EXPERIMENTS
    if constexpr (LK == LK_SYM_OTF || LK == LK_ASYM_OTF) {
        if (variant == 6) return launch_cpo<Real, D, LK, MASS, RED>(a, st);
    }
#endif
    if constexpr (D <= 8) {
        if (variant == 7) return launch_bulk<Real, D, LK, MASS, RED>(a, st, BulkTuning{ lt.bulk_rows, lt.bulk_stages, lt.bulk_ctas });
        if constexpr ((2 * D) % RPV == 0 && (D >= 6 || LK == LK_SYM_OTF || LK == LK_ASYM_OTF)) {
            if (variant == 8) return launch_bulk<Real, D, LK, MASS, RED, 2>(a, st, BulkTuning{ lt.bulk_rows, lt.bulk_stages, lt.bulk_ctas });
        }
    }
#ifdef HR_BUILD_EXPERIMENTS
    if constexpr (D <= 8 && (2 * D) % RPV == 0) {
        if (variant == 11) return launch_loop<Real, D, LK, MASS, RED>(block, a, st);
    }
#endif
    if constexpr (D <= 4) {
        const BulkTuning bt{ lt.bulk_rows, lt.bulk_stages, lt.bulk_ctas };
        if (variant == 9) return launch_bulkx<Real, D, LK, MASS, RED, 1>(a, st, bt, lt.bulk_strip);
        if constexpr ((2 * D) % RPV == 0) {
            if (variant == 10) return launch_bulkx<Real, D, LK, MASS, RED, 2>(a, st, bt, lt.bulk_strip);
        }
    }
    if constexpr (D > 8) {
        if (variant == 0) return launch_one<Real, D, LK, 1, MASS, RED, LD_STREAM, LD_DEFAULT, ST_DEFAULT>(block, a, st);
    } else
    switch (variant) {
    case 0: return launch_one<Real, D, LK, 1, MASS, RED, LD_STREAM, LD_DEFAULT, ST_DEFAULT>(block, a, st);
    case 1: return launch_one<Real, D, LK, 1, MASS, RED, LD_STREAM_EF, LD_KEEP, ST_STREAM>(block, a, st);
    case 2:
        if constexpr (PAIR_OK) return launch_one<Real, D, LK, 2, MASS, RED, LD_STREAM, LD_DEFAULT, ST_DEFAULT>(block, a, st);
        break;
    case 3:
        if constexpr (PAIR_OK) return launch_one<Real, D, LK, 2, MASS, RED, LD_STREAM_EF, LD_KEEP, ST_STREAM>(block, a, st);
        break;
#ifdef HR_BUILD_EXPERIMENTS
    case 4: return launch_one<Real, D, LK, 1, MASS, RED, LD_DEFAULT, LD_DEFAULT, ST_DEFAULT>(block, a, st);
    case 5:
        if constexpr (PfGeom<Real, D, LK>::smem_bytes(64) <= kMaxDynSmem) return launch_pf<Real, D, LK, MASS, RED>(block, a, st);
        break;
#endif
    default: break;
    }
    set_error("dphi variant %d not available for d_R=%d, %s", variant, D, sizeof(Real) == 8 ? "fp64" : "fp32");
    return HR_EUNSUPPORTED;
}

template <typename Real, int D, int LK>
hr_status launch_dphi_t(int variant, const LaunchTune &lt, const DphiArgs &a, cudaStream_t st)
{
    const int block = lt.block;
    if (a.site_mode != 0) {
        // fused site-diagonal matrix: the `site` / `site_ef` kernels only, complex-link kinds with a clover field
        if constexpr ((LK == LK_COMPLEX || LK == LK_REAL) && D <= 8) {
            if (a.site_mode == 1 && a.self && !a.red_result) {
                if (variant == 0) return launch_one<Real, D, LK, 1, true, false, LD_STREAM, LD_DEFAULT, ST_DEFAULT, 1>(block, a, st);
                if (variant == 1) return launch_one<Real, D, LK, 1, true, false, LD_STREAM_EF, LD_KEEP, ST_STREAM, 1>(block, a, st);
            }
            if (a.site_mode == 2 && !a.self) {
                if (variant == 0) return launch_one<Real, D, LK, 1, false, false, LD_STREAM, LD_DEFAULT, ST_DEFAULT, 2>(block, a, st);
                if (variant == 1) return launch_one<Real, D, LK, 1, false, false, LD_STREAM_EF, LD_KEEP, ST_STREAM, 2>(block, a, st);
            }
        }
        set_error("fused site matrix: not available for this kernel variant / link kind");
        return HR_EUNSUPPORTED;
    }
    if (a.self && a.red_result) return launch_variant<Real, D, LK, true, true>(variant, lt, a, st);
    if (a.self) return launch_variant<Real, D, LK, true, false>(variant, lt, a, st);
    return launch_variant<Real, D, LK, false, false>(variant, lt, a, st);
}

template <typename Real, int D, int LK> bool dphi_variant_ok_t(int variant)
{
    constexpr int RPV = 16 / (int)sizeof(Real);
    if (variant < 0 || variant >= DPHI_NVARIANTS) return false;
    if (variant == 6) return LK == LK_COMPLEX || LK == LK_REAL || (kExperiments && (LK == LK_SYM_OTF || LK == LK_ASYM_OTF));
    if (variant == 7) return D <= 8;   // whether a tile can be aligned on THIS lattice is decided at launch (bulk_geometry)
    if (variant == 8) return D <= 8 && (2 * D) % RPV == 0 && (D >= 6 || LK == LK_SYM_OTF || LK == LK_ASYM_OTF);
    if (variant == 9) return D <= 4;
    if (variant == 10) return D <= 4 && (2 * D) % RPV == 0;
    if (variant == 11) return kExperiments && D <= 8 && (2 * D) % RPV == 0;
    if (D > 8) return variant == 0;
    if ((variant == 2 || variant == 3) && ((2 * D) % RPV != 0 || !(D >= 6 || kExperiments))) return false;
    if (variant == 4 || variant == 5) {
#ifdef HR_BUILD_EXPERIMENTS
        return variant == 4 || PfGeom<Real, D, LK>::smem_bytes(64) <= kMaxDynSmem;
#else
        return false;
#endif
    }
    return true;
}

// can the bulk kernel tile this lattice (alignment of the tail planes, Zh <= 128)?
template <typename Real, int D, int LK> bool dphi_bulk_ok_t(const DphiArgs &a, int ks)
{
    if constexpr (D <= 8) {
        BulkArgs g;
        return bulk_geometry<Real, D, LK>(a, g, kMaxDynSmem - 1024, 0, 0, ks == 1 ? BulkGeom<Real, D, LK>::MAXN : 112);
    } else return false;
}

template <typename Real, int D, int LK> hr_status launch_halo_t(bool pack, int mu, const HaloArgs &a, cudaStream_t st)
{
    const unsigned grid = (unsigned)((a.nface + 127) / 128);
#define HR_HALO_MU(M)                                                                                     \
    case M:                                                                                               \
        if (pack) halo_pack_kernel<Real, D, LK, M><<<grid, 128, 0, st>>>(a);                              \
        else halo_apply_kernel<Real, D, LK, M><<<grid, 128, 0, st>>>(a);                                  \
        break;
    switch (mu) {
        HR_HALO_MU(0) HR_HALO_MU(1) HR_HALO_MU(2) HR_HALO_MU(3)
    default: set_error("halo kernels: direction %d", mu); return HR_EINVAL;
    }
#undef HR_HALO_MU
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) {
        set_error("halo %s kernel launch failed: %s", pack ? "pack" : "apply", cudaGetErrorString(e));
        return HR_ECUDA;
    }
    return HR_OK;
}

// pack == true: the messages of all split directions; false: their face terms added to out (halo_kernel.cuh); mu ascending
template <typename Real, int D, int LK> hr_status launch_halo_multi_t(bool pack, const HaloArgs *a, const int *mu, int ndir, cudaStream_t st)
{
    HaloMultiArgs g;
    g.ndir = ndir;
    g.first[0] = 0;
    for (int m = 0; m < 4; ++m) g.slot[m] = -1;
    for (int k = 0; k < ndir; ++k) {
        g.a[k] = a[k];
        g.mu[k] = mu[k];
        g.slot[mu[k]] = k;
        g.first[k + 1] = g.first[k] + (unsigned)((a[k].nface + 127) / 128);
    }
    for (int k = ndir; k < 4; ++k) { g.a[k] = a[0]; g.mu[k] = 0; g.first[k + 1] = g.first[ndir]; }
    if (pack) halo_pack_multi_kernel<Real, D, LK><<<g.first[ndir], 128, 0, st>>>(g);
    else halo_apply_multi_kernel<Real, D, LK><<<g.first[ndir], 128, 0, st>>>(g);
    count_launch();
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { set_error("halo multi-direction %s launch failed: %s", pack ? "pack" : "apply", cudaGetErrorString(e)); return HR_ECUDA; }
    return HR_OK;
}

#define HR_DPHI_INSTANCE(Real, D, LK)                                                                    \
    template hr_status launch_dphi_t<Real, D, LK>(int, const LaunchTune &, const DphiArgs &, cudaStream_t); \
    template bool dphi_variant_ok_t<Real, D, LK>(int);                                                    \
    template bool dphi_bulk_ok_t<Real, D, LK>(const DphiArgs &, int);                                                \
    template hr_status launch_halo_t<Real, D, LK>(bool, int, const HaloArgs &, cudaStream_t);             \
    template hr_status launch_halo_multi_t<Real, D, LK>(bool, const HaloArgs *, const int *, int, cudaStream_t);

} // namespace hr
