// Register-resident fused FFT kernels (the fast path of SURVEY S1/S3/S4/S6 when every axis length is a two-stage
// plan N = R1*R2 and one (y,z) plane fits in shared memory).
//
//   plane_kernel  one CTA = one x-plane of one packed grid: the z and y transforms of the plane in one visit.
//                 Each thread holds the R elements of one butterfly in registers; global memory is read straight
//                 into the first butterfly and written straight out of the last one; shared memory only carries
//                 the three exchanges between stages (96 bytes per point instead of 2 x 96 for two staged passes).
//                 The pointwise neighbours are fused into the load / store functors (pair product phi_v*phi_v',
//                 re/im packing of two real functions, split + scale into the chunked real-space batches).
//   xpass_kernel  one CTA = NX x W tile of x-columns: forward, inverse, or forward * Coulomb table * inverse
//                 (tau_vv' = C[phi_v phi_v']) with the last forward stage, the table multiply and
//                 the first inverse stage done in the same registers (two exchanges, 64 bytes per point).
//
// Orders are those of fft_core.cuh: forward = decimation in frequency (natural in, digit-reversed out), inverse =
// decimation in time, so both kernels agree with the general pass kernels and with the host tables (plan.cpp).
// Twiddles w_r = exp(-2 pi i * i*r / N) of a thread's fixed residue i live in registers.
#pragma once
#include "fft_steps.cuh"

namespace tddft {

template <int N> struct Two {   // two-stage view of Plan<N>
    static constexpr int R1 = Plan<N>::R1, R2 = Plan<N>::R2;
    static constexpr bool ok = (Plan<N>::R3 == 1) && (R2 > 1);
    static constexpr int PADP = (R2 % 2 == 0) ? R2 : 0;                 // pad one slot every R2 elements when R2 is even
    static constexpr int NP = PADP ? N + N / PADP : N;                  // padded pencil length
    static constexpr int PITCH = (NP % 2 == 0) ? NP + 1 : NP;           // odd pitch: strided (y) accesses hit distinct banks
    __host__ __device__ static constexpr int pad(int e) { return PADP ? e + e / PADP : e; }
};

// twiddles of residue i: w[r] = tw[i*r], r = 1..R1-1 (w[0] unused)
template <int R1> __device__ __forceinline__ void load_twiddles(const cplx* __restrict__ tw, int i, cplx (&w)[R1]) {
    w[0] = make_double2(1.0, 0.0);
#pragma unroll
    for (int r = 1; r < R1; ++r) w[r] = __ldg(&tw[i * r]);
}

// ---- bound load / store functors: per-CTA state resolved once ----------------------------------------------
struct BLoadWork { const cplx* g; __device__ __forceinline__ cplx operator()(long idx) const { return g[idx]; } };
struct BStoreWork { cplx* g; __device__ __forceinline__ void operator()(long idx, cplx v) const { g[idx] = v; } };
struct BLoadPair {
    const double *a0, *a1, *b0, *b1;   // re = a0*a1, im = b0*b1 (b0 null: im = 0)
    __device__ __forceinline__ cplx operator()(long idx) const {
        const double re = __ldg(a0 + idx) * __ldg(a1 + idx);
        const double im = b0 ? __ldg(b0 + idx) * __ldg(b1 + idx) : 0.0;
        return make_double2(re, im);
    }
};
struct BLoadPack2 {
    const double* s0; const double* s1; BatchLayout lay; long f; bool has_im; double scale;
    __device__ __forceinline__ cplx operator()(long idx) const {
        const long o0 = lay(f, idx);
        double re = s0[o0]; if (s1) re += s1[o0];
        double im = 0.0;
        if (has_im) { const long o1 = o0 + lay.next(); im = s0[o1]; if (s1) im += s1[o1]; }
        return make_double2(re * scale, im * scale);
    }
};
struct BStoreSplit2 {
    double* dst; BatchLayout lay; long f; bool has_im; double scale;
    __device__ __forceinline__ void operator()(long idx, cplx v) const {
        const long o0 = lay(f, idx);
        dst[o0] = v.x * scale;
        if (has_im) dst[o0 + lay.next()] = v.y * scale;
    }
};
__device__ __forceinline__ BLoadWork bind(const LoadWork& l, int b) { return BLoadWork{l.work + (long)b * l.nr}; }
__device__ __forceinline__ BStoreWork bind(const StoreWork& s, int b) { return BStoreWork{s.work + (long)b * s.nr}; }
__device__ __forceinline__ BLoadPair bind(const LoadPair& l, int b) {
    const int2 p0 = l.pairs[2 * b];
    BLoadPair r{l.phi + (long)p0.x * l.nr, l.phi + (long)p0.y * l.nr, nullptr, nullptr};
    if (2 * b + 1 < l.npairs) { const int2 p1 = l.pairs[2 * b + 1]; r.b0 = l.phi + (long)p1.x * l.nr; r.b1 = l.phi + (long)p1.y * l.nr; }
    return r;
}
__device__ __forceinline__ BLoadPack2 bind(const LoadPack2& l, int b) { return BLoadPack2{l.src0, l.src1, l.lay, 2L * b, 2 * b + 1 < l.nfun, l.scale}; }
__device__ __forceinline__ BStoreSplit2 bind(const StoreSplit2& s, int b) { return BStoreSplit2{s.dst, s.lay, 2L * b, 2 * b + 1 < s.nfun, s.scale}; }

// ---- plane kernel -------------------------------------------------------------------------------------------
// grid = (NX planes, batch).  Flat index of (x, y, z) inside a grid: (x*NY + y)*NZ + z.
template <int NY, int NZ, int NTHR, int MINB, bool INV, class Load, class Store>
__global__ void __launch_bounds__(NTHR, MINB) plane_kernel(Load ld, Store st, const cplx* __restrict__ twy_g, const cplx* __restrict__ twz_g) {
    using TY = Two<NY>; using TZ = Two<NZ>;
    constexpr int R1y = TY::R1, R2y = TY::R2, R1z = TZ::R1, R2z = TZ::R2;
    constexpr int PITCH = TZ::PITCH;
    constexpr bool ZFIX = (NTHR % R2z == 0), YFIX = (NTHR % R2y == 0);     // residue i = tid % R2 is the same in every round
    extern __shared__ cplx sm[];
    const int tid = threadIdx.x;
    const long pbase = (long)blockIdx.x * NY * NZ;
    const auto L = bind(ld, (int)blockIdx.y);
    const auto S = bind(st, (int)blockIdx.y);
    cplx wz[R1z], wy[R1y];
    if (ZFIX) load_twiddles<R1z>(twz_g, tid % R2z, wz);
    if (YFIX) load_twiddles<R1y>(twy_g, tid % R2y, wy);

    if constexpr (!INV) {
        // z stage 1 (radix R1z, twiddle after): global -> registers -> shared
        for (int t = tid; t < NY * R2z; t += NTHR) {
            const int y = t / R2z, i = t - y * R2z;
            if (!ZFIX) load_twiddles<R1z>(twz_g, i, wz);
            cplx x[R1z];
#pragma unroll
            for (int r = 0; r < R1z; ++r) x[r] = L(pbase + y * NZ + i + R2z * r);
            Dft<R1z, false>::run(x);
            cplx* row = sm + y * PITCH;
            row[TZ::pad(i)] = x[0];
#pragma unroll
            for (int k = 1; k < R1z; ++k) row[TZ::pad(i + R2z * k)] = cmul(x[k], wz[k]);
        }
        __syncthreads();
        // z stage 2 (radix R2z on blocks of R2z consecutive positions), in place
        for (int t = tid; t < NY * R1z; t += NTHR) {
            const int y = t / R1z, k1 = t - y * R1z;
            cplx* blk = sm + y * PITCH + TZ::pad(k1 * R2z);
            cplx x[R2z];
#pragma unroll
            for (int i = 0; i < R2z; ++i) x[i] = blk[i];
            Dft<R2z, false>::run(x);
#pragma unroll
            for (int i = 0; i < R2z; ++i) blk[i] = x[i];
        }
        __syncthreads();
        // y stage 1 (radix R1y, twiddle after): lanes run over the residue i, the odd pitch keeps them on distinct banks
        for (int t = tid; t < NZ * R2y; t += NTHR) {
            const int zp = t / R2y, i = t - zp * R2y;
            if (!YFIX) load_twiddles<R1y>(twy_g, i, wy);
            cplx* col = sm + TZ::pad(zp) + i * PITCH;
            cplx x[R1y];
#pragma unroll
            for (int r = 0; r < R1y; ++r) x[r] = col[r * R2y * PITCH];
            Dft<R1y, false>::run(x);
            col[0] = x[0];
#pragma unroll
            for (int k = 1; k < R1y; ++k) col[k * R2y * PITCH] = cmul(x[k], wy[k]);
        }
        __syncthreads();
        // y stage 2 (radix R2y): shared -> registers -> global, lanes run over z (coalesced rows)
        for (int t = tid; t < NZ * R1y; t += NTHR) {
            const int k1 = t / NZ, zp = t - k1 * NZ;
            const cplx* col = sm + TZ::pad(zp) + (k1 * R2y) * PITCH;
            cplx x[R2y];
#pragma unroll
            for (int i = 0; i < R2y; ++i) x[i] = col[i * PITCH];
            Dft<R2y, false>::run(x);
#pragma unroll
            for (int k = 0; k < R2y; ++k) S(pbase + (long)(k1 * R2y + k) * NZ + zp, x[k]);
        }
    } else {
        // y inverse stage R2y: global -> registers -> shared
        for (int t = tid; t < NZ * R1y; t += NTHR) {
            const int k1 = t / NZ, zp = t - k1 * NZ;
            cplx x[R2y];
#pragma unroll
            for (int i = 0; i < R2y; ++i) x[i] = L(pbase + (long)(k1 * R2y + i) * NZ + zp);
            Dft<R2y, true>::run(x);
            cplx* col = sm + TZ::pad(zp) + (k1 * R2y) * PITCH;
#pragma unroll
            for (int i = 0; i < R2y; ++i) col[i * PITCH] = x[i];
        }
        __syncthreads();
        // y inverse stage R1y (conjugate twiddle before the butterfly), in place
        for (int t = tid; t < NZ * R2y; t += NTHR) {
            const int zp = t / R2y, i = t - zp * R2y;
            if (!YFIX) load_twiddles<R1y>(twy_g, i, wy);
            cplx* col = sm + TZ::pad(zp) + i * PITCH;
            cplx x[R1y];
            x[0] = col[0];
#pragma unroll
            for (int k = 1; k < R1y; ++k) x[k] = cmulc(col[k * R2y * PITCH], wy[k]);
            Dft<R1y, true>::run(x);
#pragma unroll
            for (int r = 0; r < R1y; ++r) col[r * R2y * PITCH] = x[r];
        }
        __syncthreads();
        // z inverse stage R2z, in place
        for (int t = tid; t < NY * R1z; t += NTHR) {
            const int y = t / R1z, k1 = t - y * R1z;
            cplx* blk = sm + y * PITCH + TZ::pad(k1 * R2z);
            cplx x[R2z];
#pragma unroll
            for (int i = 0; i < R2z; ++i) x[i] = blk[i];
            Dft<R2z, true>::run(x);
#pragma unroll
            for (int i = 0; i < R2z; ++i) blk[i] = x[i];
        }
        __syncthreads();
        // z inverse stage R1z: shared -> registers -> global (natural order)
        for (int t = tid; t < NY * R2z; t += NTHR) {
            const int y = t / R2z, i = t - y * R2z;
            if (!ZFIX) load_twiddles<R1z>(twz_g, i, wz);
            const cplx* row = sm + y * PITCH;
            cplx x[R1z];
            x[0] = row[TZ::pad(i)];
#pragma unroll
            for (int k = 1; k < R1z; ++k) x[k] = cmulc(row[TZ::pad(i + R2z * k)], wz[k]);
            Dft<R1z, true>::run(x);
#pragma unroll
            for (int r = 0; r < R1z; ++r) S(pbase + y * NZ + i + R2z * r, x[r]);
        }
    }
}

// ---- x pass kernel ------------------------------------------------------------------------------------------
// Columns along x (element stride `inner` = NY*NZ) of `batch` packed grids.  CTA tile = NX x XW columns; thread
// (c = tid % XW, g = tid / XW) owns residue i = g in the radix-R1 stage and block k1 = g in the radix-R2 stage, so
// its twiddles and (SM_CONV) its R2 Coulomb-table values stay in registers while the CTA walks over the batch.
// grid = (column tiles, batch groups): CTA (tx, gy) handles grids gy, gy + gridDim.y, ...
constexpr int XW = 32;
template <int NX> struct XCfg {
    static constexpr int R1 = Two<NX>::R1, R2 = Two<NX>::R2;
    static constexpr int G = R1 > R2 ? R1 : R2;
    static constexpr int NTHR = G * XW;
    static constexpr size_t SMEM = sizeof(cplx) * NX * XW;
};
template <int NX, int MODE>
__global__ void __launch_bounds__(XCfg<NX>::NTHR, 2) xpass_kernel(cplx* __restrict__ work, long inner, long nr, int batch,
                                                                 const cplx* __restrict__ tw_g, const double* __restrict__ ktab) {
    constexpr int R1 = XCfg<NX>::R1, R2 = XCfg<NX>::R2;
    extern __shared__ cplx sm[];
    const int tid = threadIdx.x, c = tid % XW, g = tid / XW;
    const long col = (long)blockIdx.x * XW + c;
    const bool live = col < inner;
    cplx w[R1];
    load_twiddles<R1>(tw_g, g < R2 ? g : 0, w);
    double kt[R2];
    if (MODE == SM_CONV) {
#pragma unroll
        for (int k = 0; k < R2; ++k) kt[k] = (live && g < R1) ? __ldg(ktab + (long)(g * R2 + k) * inner + col) : 0.0;
    }
    for (int b = blockIdx.y; b < batch; b += gridDim.y) {
        cplx* gcol = work + (long)b * nr + col;
        if (MODE == SM_FWD || MODE == SM_CONV) {
            if (g < R2) {       // stage R1 forward: rows g + R2*r
                cplx x[R1];
#pragma unroll
                for (int r = 0; r < R1; ++r) x[r] = live ? gcol[(long)(g + R2 * r) * inner] : make_double2(0.0, 0.0);
                Dft<R1, false>::run(x);
                sm[g * XW + c] = x[0];
#pragma unroll
                for (int k = 1; k < R1; ++k) sm[(g + R2 * k) * XW + c] = cmul(x[k], w[k]);
            }
            __syncthreads();
        }
        if (g < R1) {           // block g: rows g*R2 + i
            cplx x[R2];
            if (MODE == SM_INV) {
#pragma unroll
                for (int i = 0; i < R2; ++i) x[i] = live ? gcol[(long)(g * R2 + i) * inner] : make_double2(0.0, 0.0);
            } else {
#pragma unroll
                for (int i = 0; i < R2; ++i) x[i] = sm[(g * R2 + i) * XW + c];
                Dft<R2, false>::run(x);
            }
            if (MODE == SM_FWD) {
                if (live) {
#pragma unroll
                    for (int k = 0; k < R2; ++k) gcol[(long)(g * R2 + k) * inner] = x[k];
                }
            } else {
                if (MODE == SM_CONV) {
#pragma unroll
                    for (int k = 0; k < R2; ++k) { x[k].x *= kt[k]; x[k].y *= kt[k]; }
                }
                Dft<R2, true>::run(x);
#pragma unroll
                for (int i = 0; i < R2; ++i) sm[(g * R2 + i) * XW + c] = x[i];
            }
        }
        if (MODE != SM_FWD) {
            __syncthreads();
            if (g < R2) {       // stage R1 inverse: conjugate twiddle, butterfly, natural order out
                cplx x[R1];
                x[0] = sm[g * XW + c];
#pragma unroll
                for (int k = 1; k < R1; ++k) x[k] = cmulc(sm[(g + R2 * k) * XW + c], w[k]);
                Dft<R1, true>::run(x);
                if (live) {
#pragma unroll
                    for (int r = 0; r < R1; ++r) gcol[(long)(g + R2 * r) * inner] = x[r];
                }
            }
        }
        __syncthreads();        // the tile is reused by the next grid of the batch
    }
}

}  // namespace tddft
