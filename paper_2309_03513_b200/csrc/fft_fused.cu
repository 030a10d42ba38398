// Instantiations and host dispatch of the fused FFT kernels (fft_fused.cuh) for the grid shapes of the BASELINE.json
// configurations that fit the fast path; every other shape runs the general pass kernels (fft_steps.cuh).
#include <type_traits>
#include "fft_fused.cuh"
#include "fft_cluster.cuh"

namespace tddft {

// (NY, NZ, threads per CTA, CTAs per SM the registers are budgeted for)
#define TD_FOR_EACH_PLANE(X) X(72, 72, 216, 2) X(48, 48, 96, 5) X(24, 24, 96, 8) X(18, 20, 96, 8) X(96, 100, 360, 1) X(108, 108, 324, 1)
#define TD_FOR_EACH_XLEN(X) X(72) X(48) X(24) X(12) X(96) X(108) X(128)
// planes held by a cluster of two CTAs (fft_cluster.cuh): (NY, NZ, threads per CTA, CTAs per SM)
#define TD_FOR_EACH_CPLANE(X) X(128, 128, 512, 1) X(96, 100, 256, 2) X(108, 108, 256, 2)

// Launch policy, fixed after the round-1 measurements (profiles/r01g_summary.md, r01i_summary.md): persistent grids that walk
// the units plane-major; L2 prefetch of the CTA's next work-grid plane (inverse kernels) but not of orbital planes (they are
// shared with the units running now); evict-first L2 policy on the work-grid / tau / a(r) streams.
constexpr int kStreamHint = 1;
// launch with programmatic stream serialization (see pdl_wait in fft_fused.cuh)
template <class... KArgs, class... Args>
static cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, unsigned block, size_t smem, cudaStream_t s, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}
template <int NY, int NZ, int NTHR, int MINB, bool INV, bool DB1, bool DB2, class Load, class Store>
static cudaError_t plane_launch2(Load ld, Store st, const ZArgs& a, cudaStream_t s) {
    static_assert(Two<NY>::ok && Two<NZ>::ok, "fused plane kernel needs two-stage plans");
    const size_t smem = sizeof(cplx) * (size_t)NY * Two<NZ>::PITCH;
    auto kern = plane_kernel<NY, NZ, NTHR, MINB, INV, DB1, DB2, Load, Store>;
    static int resident[kMaxDevices] = {0};                   // CTAs the device holds at once; 0 = attributes not set yet
    const int dev = current_device();
    if (!resident[dev]) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        int sms = 0, per_sm = 0;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NTHR, smem);
        resident[dev] = sms * (per_sm > 0 ? per_sm : 1);
    }
    const int nx = (int)(a.npencils / NY), nunits = nx * a.batch;
    const int grid = nunits < resident[dev] ? nunits : resident[dev];
    const int l2pf = std::is_same<Load, LoadWorkC>::value ? 1 : 0;
    return launch_pdl(kern, dim3(grid), NTHR, smem, s, ld, st, nx, nunits, l2pf, a.tw2, a.tw);
}
template <int NY, int NZ, int NTHR, int MINB, bool INV, class Load, class Store>
static cudaError_t plane_launch(Load ld, Store st, const ZArgs& a, cudaStream_t s) {
    // double-buffered rounds (DB1 / DB2 of plane_kernel) measured slower on B200 (register pressure): both off
    return plane_launch2<NY, NZ, NTHR, MINB, INV, false, false>(ld, st, a, s);
}
template <int NY, int NZ, int NTHR, int MINB>
static cudaError_t plane_dispatch(bool inverse, int lkind, int skind, const ZArgs& a, cudaStream_t s) {
    const int hint = kStreamHint;
    LoadWorkC lw{a.work, a.wstride, a.cmap, a.ncols, a.whint};
    StoreWorkC sw{a.work, a.wstride, a.cmap, a.ncols, a.whint};
    const BatchLayout lay{a.chunked, a.fbase, a.ftotal * CHUNK, a.nr};
    if (!inverse) {
        if (lkind == ZL_PAIR) return plane_launch<NY, NZ, NTHR, MINB, false>(LoadPair{a.phi, a.phi2 ? a.phi2 : a.phi, a.pairs, a.npairs, a.nr}, sw, a, s);
        if (lkind == ZL_PACK2) return plane_launch<NY, NZ, NTHR, MINB, false>(LoadPack2{a.src0, a.src1, a.nfun, lay, a.lscale}, sw, a, s);
        return cudaErrorInvalidValue;
    }
    if (skind == ZS_SPLIT2) return plane_launch<NY, NZ, NTHR, MINB, true>(lw, StoreSplit2{a.dst, a.nfun, lay, a.sscale, hint, a.slots}, a, s);
    return cudaErrorInvalidValue;
}

template <int NY, int NZ, int NTHR, int MINB, bool INV, class Load, class Store>
static cudaError_t cplane_launch(Load ld, Store st, const ZArgs& a, cudaStream_t s) {
    static_assert(Two<NY>::ok && Two<NZ>::ok, "cluster plane kernel needs two-stage plans");
    const size_t smem = sizeof(cplx) * (size_t)(NY / 2) * Two<NZ>::PITCH;
    auto kern = plane_cluster_kernel<NY, NZ, NTHR, MINB, INV, Load, Store>;
    cudaLaunchConfig_t cfg = {};
    cfg.blockDim = dim3(NTHR); cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 2;
    static int resident[kMaxDevices] = {0};                   // clusters the device holds at once
    const int dev = current_device();
    if (!resident[dev]) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        int sms = 0; cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cfg.gridDim = dim3(2 * sms * MINB);
        int ncl = 0;
        e = cudaOccupancyMaxActiveClusters(&ncl, kern, &cfg);
        if (e != cudaSuccess || ncl < 1) { cudaGetLastError(); ncl = sms * MINB / 2; }
        resident[dev] = ncl;
    }
    const int nx = (int)(a.npencils / NY), nunits = nx * a.batch;
    cfg.gridDim = dim3(2 * (unsigned)(nunits < resident[dev] ? nunits : resident[dev]));
    return cudaLaunchKernelEx(&cfg, kern, ld, st, nx, nunits, a.tw2, a.tw);
}
template <int NY, int NZ, int NTHR, int MINB>
static cudaError_t cplane_dispatch(bool inverse, int lkind, int skind, const ZArgs& a, cudaStream_t s) {
    LoadWorkC lw{a.work, a.wstride, a.cmap, a.ncols, a.whint};
    StoreWorkC sw{a.work, a.wstride, a.cmap, a.ncols, a.whint};
    const BatchLayout lay{a.chunked, a.fbase, a.ftotal * CHUNK, a.nr};
    if (!inverse) {
        if (lkind == ZL_PAIR) return cplane_launch<NY, NZ, NTHR, MINB, false>(LoadPair{a.phi, a.phi2 ? a.phi2 : a.phi, a.pairs, a.npairs, a.nr}, sw, a, s);
        if (lkind == ZL_PACK2) return cplane_launch<NY, NZ, NTHR, MINB, false>(LoadPack2{a.src0, a.src1, a.nfun, lay, a.lscale}, sw, a, s);
        return cudaErrorInvalidValue;
    }
    if (skind == ZS_SPLIT2) return cplane_launch<NY, NZ, NTHR, MINB, true>(lw, StoreSplit2{a.dst, a.nfun, lay, a.sscale, kStreamHint, a.slots}, a, s);
    return cudaErrorInvalidValue;
}

template <int NX>
static cudaError_t xpass_generic_launch(int mode, const SArgs& a, cudaStream_t s) {
    constexpr size_t smem = XGCfg<NX>::SMEM;
    static int resident_d[kMaxDevices] = {0};
    const int dev = current_device();
    if (!resident_d[dev]) {
        cudaError_t e = cudaFuncSetAttribute(xpass_generic_kernel<NX, SM_FWD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(xpass_generic_kernel<NX, SM_INV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(xpass_generic_kernel<NX, SM_CONV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        int sms = 0, per_sm = 0;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, xpass_generic_kernel<NX, SM_CONV>, XGCfg<NX>::NTHR, smem);
        resident_d[dev] = sms * (per_sm > 0 ? per_sm : 1);
    }
    const unsigned tiles = (unsigned)((a.inner + XGCfg<NX>::XWG - 1) / XGCfg<NX>::XWG);
    int gy = 1;      // at least 3 waves of the resident CTAs (or one grid per CTA)
    while (gy < a.batch && (long)tiles * gy < 3L * resident_d[dev]) ++gy;
    dim3 grid(tiles, (unsigned)gy);
    constexpr int NT = XGCfg<NX>::NTHR;
    if (mode == SM_FWD) return launch_pdl(xpass_generic_kernel<NX, SM_FWD>, grid, NT, smem, s, a.work, a.inner, a.nr, a.batch, a.tw, a.ktab, a.whint);
    if (mode == SM_INV) return launch_pdl(xpass_generic_kernel<NX, SM_INV>, grid, NT, smem, s, a.work, a.inner, a.nr, a.batch, a.tw, a.ktab, a.whint);
    return launch_pdl(xpass_generic_kernel<NX, SM_CONV>, grid, NT, smem, s, a.work, a.inner, a.nr, a.batch, a.tw, a.ktab, a.whint);
}
template <int NX>
static cudaError_t xpass_launch(int mode, const SArgs& a, cudaStream_t s) {
    static_assert(Two<NX>::ok, "fused x pass needs a two-stage plan");
    if constexpr (XCfg<NX>::G > 12) return xpass_generic_launch<NX>(mode, a, s);
    else {
    constexpr size_t smem = XCfg<NX>::SMEM;
    static int resident_d[kMaxDevices] = {0};
    const int dev = current_device();
    if (!resident_d[dev]) {
        cudaError_t e = cudaFuncSetAttribute(xpass_kernel<NX, SM_FWD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(xpass_kernel<NX, SM_INV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(xpass_kernel<NX, SM_CONV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        int sms = 0, per_sm = 0;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, xpass_kernel<NX, SM_CONV>, XCfg<NX>::NTHR, smem);
        resident_d[dev] = sms * (per_sm > 0 ? per_sm : 1);
    }
    const int resident = resident_d[dev];
    // batch groups: enough CTAs for ~6 waves of the resident set, each CTA keeps its twiddles and Coulomb-table values
    // in registers while it walks over its grids
    const unsigned tiles = (unsigned)((a.inner + XW - 1) / XW);
    int gy = a.batch, best_gy = a.batch; double best = 0.0;
    for (gy = 1; gy <= a.batch; ++gy) {
        if ((long)tiles * gy < 3L * resident && gy < a.batch) continue;      // at least 3 waves (or one grid per CTA)
        const long ctas = (long)tiles * gy, waves = (ctas + resident - 1) / resident;
        const int per = (a.batch + gy - 1) / gy;                              // grids per CTA: imbalance when batch % gy != 0
        const double eff = (double)ctas / (double)(waves * resident) * (double)a.batch / (double)(per * gy);
        if (eff > best + 1e-9) { best = eff; best_gy = gy; }
    }
    dim3 grid(tiles, (unsigned)best_gy);
    constexpr int NT = XCfg<NX>::NTHR;
    if (mode == SM_FWD) return launch_pdl(xpass_kernel<NX, SM_FWD>, grid, NT, smem, s, a.work, a.inner, a.nr, a.batch, a.tw, a.ktab, a.whint);
    if (mode == SM_INV) return launch_pdl(xpass_kernel<NX, SM_INV>, grid, NT, smem, s, a.work, a.inner, a.nr, a.batch, a.tw, a.ktab, a.whint);
    return launch_pdl(xpass_kernel<NX, SM_CONV>, grid, NT, smem, s, a.work, a.inner, a.nr, a.batch, a.tw, a.ktab, a.whint);
    }
}

bool fused_supported(const int* n) {
    bool px = false, pl = false;
#define X(N) if (n[0] == N) px = true;
    TD_FOR_EACH_XLEN(X)
#undef X
#define X(NY, NZ, T, B) if (n[1] == NY && n[2] == NZ) pl = true;
    TD_FOR_EACH_PLANE(X)
    TD_FOR_EACH_CPLANE(X)
#undef X
    return px && pl;
}
cudaError_t launch_plane(int ny, int nz, bool inverse, int lkind, int skind, const ZArgs& a, cudaStream_t st) {
    // a.cluster: prefer the two-CTA cluster kernel where the shape has both (the only one for 128 x 128)
#define X(NY, NZ, T, B) if (a.cluster && ny == NY && nz == NZ) return cplane_dispatch<NY, NZ, T, B>(inverse, lkind, skind, a, st);
    TD_FOR_EACH_CPLANE(X)
#undef X
#define X(NY, NZ, T, B) if (ny == NY && nz == NZ) return plane_dispatch<NY, NZ, T, B>(inverse, lkind, skind, a, st);
    TD_FOR_EACH_PLANE(X)
#undef X
#define X(NY, NZ, T, B) if (ny == NY && nz == NZ) return cplane_dispatch<NY, NZ, T, B>(inverse, lkind, skind, a, st);
    TD_FOR_EACH_CPLANE(X)
#undef X
    return cudaErrorInvalidValue;
}
cudaError_t launch_xpass(int mode, const SArgs& a, cudaStream_t st) {
#define X(N) if (a.n == N) return xpass_launch<N>(mode, a, st);
    TD_FOR_EACH_XLEN(X)
#undef X
    return cudaErrorInvalidValue;
}

}  // namespace tddft
