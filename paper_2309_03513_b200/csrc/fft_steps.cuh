// FFT pass kernels: one 1-D transform along one axis of a batch of 3-D complex grids per launch, with the
// neighbouring pointwise steps fused into the loads/stores:
//   z pass (contiguous axis): load = orbital-pair product phi_v*phi_v' packed two pairs per complex grid
//                             (PAPER.md:230), or two real functions packed as re/im (S3, S6);
//                             store = split re/im into two real grids with a scale (S1, S3, S4).
//   strided pass (y or x axis): forward, inverse, or forward * Coulomb table * inverse in one visit (S4, S3).
// Two real grids ride as re/im of one complex transform because the Coulomb table is real and even in G.
#pragma once
#include "common.h"

namespace tddft {

struct LoadWork {
    const cplx* work; long nr;
    __device__ __forceinline__ cplx operator()(int b, long idx) const { return work[(long)b * nr + idx]; }
};
struct LoadPair {      // pair p = (x, y): density phi[x] * phi2[y] (both plain [function][nr]; K1d: phi2 = phi)
    const double* phi; const double* phi2; const int2* pairs; int npairs; long nr;
    __device__ __forceinline__ cplx operator()(int b, long idx) const {
        const int2 p0 = pairs[2 * b];
        double re = phi[(long)p0.x * nr + idx] * phi2[(long)p0.y * nr + idx];
        double im = 0.0;
        if (2 * b + 1 < npairs) {
            const int2 p1 = pairs[2 * b + 1];
            im = phi[(long)p1.x * nr + idx] * phi2[(long)p1.y * nr + idx];
        }
        return make_double2(re, im);
    }
};
struct BatchLayout {     // address of grid point idx of function f inside a batch of real functions (common.h)
    int chunked; long fbase, cstride, nr;
    __device__ __forceinline__ long operator()(long f, long idx) const {
        return chunked ? (idx >> CHUNK_LOG) * cstride + (fbase + f) * CHUNK + (idx & (CHUNK - 1)) : (fbase + f) * nr + idx;
    }
    __device__ __forceinline__ long next() const { return chunked ? CHUNK : nr; }   // offset from function f to f + 1
};
struct LoadPack2 {
    const double* src0; const double* src1; int nfun; BatchLayout lay; double scale;
    __device__ __forceinline__ cplx operator()(int b, long idx) const {
        const long o0 = lay(2 * b, idx);
        double re = src0[o0]; if (src1) re += src1[o0];
        double im = 0.0;
        if (2 * b + 1 < nfun) { const long o1 = o0 + lay.next(); im = src0[o1]; if (src1) im += src1[o1]; }
        return make_double2(re * scale, im * scale);
    }
};
struct StoreWork {
    cplx* work; long nr;
    __device__ __forceinline__ void operator()(int b, long idx, cplx v) const { work[(long)b * nr + idx] = v; }
};
struct StoreSplit2 {
    double* dst; int nfun; BatchLayout lay; double scale;
    int hint;            // fused path: L2 eviction hint of the store stream (fft_fused.cuh)
    const int* slots;    // optional: function index of packed function q is slots[q] instead of q (pair -> tau slot)
    __device__ __forceinline__ void operator()(int b, long idx, cplx v) const {
        dst[lay(slots ? slots[2 * b] : 2 * b, idx)] = v.x * scale;
        if (2 * b + 1 < nfun) dst[lay(slots ? slots[2 * b + 1] : 2 * b + 1, idx)] = v.y * scale;
    }
};

// contiguous-axis pass: CTA = PZ consecutive pencils of one grid, staged in padded shared memory
template <int N, bool INV, class Load, class Store>
__global__ void __launch_bounds__(256) zpass_kernel(Load ld, Store st, long npencils, int PZ, const cplx* __restrict__ twg) {
    extern __shared__ cplx sm[];
    constexpr int NPAD = PlanInfo<N>::NPAD;
    cplx* tw = sm + (size_t)PZ * NPAD;
    const int b = blockIdx.y;
    const long p0 = (long)blockIdx.x * PZ;
    const int np = (int)min((long)PZ, npencils - p0);
    for (int k = threadIdx.x; k < N; k += blockDim.x) tw[k] = twg[k];
    const int total = np * N;
    for (int t = threadIdx.x; t < total; t += blockDim.x) {
        const int p = t / N, z = t - p * N;
        sm[p * NPAD + pad_pos<N>(z)] = ld(b, p0 * N + t);
    }
    __syncthreads();
    fft_tile<N, INV, true>(sm, np, NPAD, 1, tw, threadIdx.x, blockDim.x, BlockSync{});
    __syncthreads();
    for (int t = threadIdx.x; t < total; t += blockDim.x) {
        const int p = t / N, z = t - p * N;
        st(b, p0 * N + t, sm[p * NPAD + pad_pos<N>(z)]);
    }
}

// strided-axis pass: CTA = N x W tile (W contiguous elements), lanes across the contiguous direction
template <int N, int MODE>
__global__ void __launch_bounds__(256) spass_kernel(cplx* __restrict__ work, long stride, long inner, long outer_stride,
                                                   long nr, int W, const cplx* __restrict__ twg,
                                                   const double* __restrict__ ktab) {
    extern __shared__ cplx sm[];
    cplx* tw = sm + (size_t)N * W;
    const long c0 = (long)blockIdx.x * W;
    const int w = (int)min((long)W, inner - c0);
    const long goff = (long)blockIdx.y * outer_stride + c0;
    cplx* base = work + (long)blockIdx.z * nr + goff;
    for (int k = threadIdx.x; k < N; k += blockDim.x) tw[k] = twg[k];
    const int total = N * w;
    for (int t = threadIdx.x; t < total; t += blockDim.x) {
        const int e = t / w, c = t - e * w;
        sm[e * W + c] = base[(long)e * stride + c];
    }
    __syncthreads();
    if (MODE == SM_FWD || MODE == SM_CONV) {
        fft_tile<N, false, false>(sm, w, 1, W, tw, threadIdx.x, blockDim.x, BlockSync{});
        __syncthreads();
    }
    if (MODE == SM_CONV) {
        const double* kt = ktab + goff;
        for (int t = threadIdx.x; t < total; t += blockDim.x) {
            const int e = t / w, c = t - e * w;
            const double k = kt[(long)e * stride + c];
            cplx v = sm[e * W + c];
            sm[e * W + c] = make_double2(v.x * k, v.y * k);
        }
        __syncthreads();
    }
    if (MODE == SM_INV || MODE == SM_CONV) {
        fft_tile<N, true, false>(sm, w, 1, W, tw, threadIdx.x, blockDim.x, BlockSync{});
        __syncthreads();
    }
    for (int t = threadIdx.x; t < total; t += blockDim.x) {
        const int e = t / w, c = t - e * w;
        base[(long)e * stride + c] = sm[e * W + c];
    }
}

template <int N> inline int zpass_pencils_per_cta() {
    int pz = (40 * 1024) / (PlanInfo<N>::NPAD * (int)sizeof(cplx));
    if (pz > 64) pz = 64;
    if (pz >= 8) pz &= ~7;
    return pz < 1 ? 1 : pz;
}
template <int N> inline int spass_tile_width() {
    int w = (32 * 1024) / (N * (int)sizeof(cplx));
    if (w > 32) w = 32;
    if (w >= 8) w &= ~7;
    return w < 1 ? 1 : w;
}

template <int N, bool INV, class Load, class Store>
cudaError_t zpass_launch(Load ld, Store st, const ZArgs& a, cudaStream_t s) {
    const int PZ = zpass_pencils_per_cta<N>();
    const size_t smem = ((size_t)PZ * PlanInfo<N>::NPAD + N) * sizeof(cplx);
    dim3 grid((unsigned)((a.npencils + PZ - 1) / PZ), (unsigned)a.batch);
    zpass_kernel<N, INV, Load, Store><<<grid, 256, smem, s>>>(ld, st, a.npencils, PZ, a.tw);
    return cudaGetLastError();
}
template <int N>
cudaError_t zpass_dispatch(bool inverse, int lkind, int skind, const ZArgs& a, cudaStream_t s) {
    LoadWork lw{a.work, a.nr};
    StoreWork sw{a.work, a.nr};
    if (!inverse) {
        // forward passes always store to the work grids
        if (lkind == ZL_PAIR) return zpass_launch<N, false>(LoadPair{a.phi, a.phi2 ? a.phi2 : a.phi, a.pairs, a.npairs, a.nr}, sw, a, s);
        if (lkind == ZL_PACK2) return zpass_launch<N, false>(LoadPack2{a.src0, a.src1, a.nfun, BatchLayout{a.chunked, a.fbase, a.ftotal * CHUNK, a.nr}, a.lscale}, sw, a, s);
        return zpass_launch<N, false>(lw, sw, a, s);
    }
    if (skind == ZS_SPLIT2) return zpass_launch<N, true>(lw, StoreSplit2{a.dst, a.nfun, BatchLayout{a.chunked, a.fbase, a.ftotal * CHUNK, a.nr}, a.sscale, 0, a.slots}, a, s);
    return zpass_launch<N, true>(lw, sw, a, s);
}
template <int N>
cudaError_t spass_dispatch(int mode, const SArgs& a, cudaStream_t s) {
    const int W = spass_tile_width<N>();
    const size_t smem = ((size_t)N * W + N) * sizeof(cplx);
    dim3 grid((unsigned)((a.inner + W - 1) / W), (unsigned)a.nouter, (unsigned)a.batch);
    if (mode == SM_FWD) spass_kernel<N, SM_FWD><<<grid, 256, smem, s>>>(a.work, a.stride, a.inner, a.outer_stride, a.nr, W, a.tw, a.ktab);
    else if (mode == SM_INV) spass_kernel<N, SM_INV><<<grid, 256, smem, s>>>(a.work, a.stride, a.inner, a.outer_stride, a.nr, W, a.tw, a.ktab);
    else spass_kernel<N, SM_CONV><<<grid, 256, smem, s>>>(a.work, a.stride, a.inner, a.outer_stride, a.nr, W, a.tw, a.ktab);
    return cudaGetLastError();
}

}  // namespace tddft
