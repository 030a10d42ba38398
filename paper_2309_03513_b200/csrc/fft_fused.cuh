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

// Programmatic dependent launch (fft_fused.cu launches these kernels with programmaticStreamSerialization): a kernel lets its
// successor in the stream start launching at once (its CTAs take the SM slots this kernel's CTAs free, and run their prologue:
// twiddles, column maps, Coulomb-table values), and waits for its predecessor to complete before it touches any work buffer.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// twiddles of residue i: w[r] = tw[i*r], r = 1..R1-1 (w[0] unused)
template <int R1> __device__ __forceinline__ void load_twiddles(const cplx* __restrict__ tw, int i, cplx (&w)[R1]) {
    w[0] = make_double2(1.0, 0.0);
#pragma unroll
    for (int r = 1; r < R1; ++r) w[r] = __ldg(&tw[i * r]);
}

// ---- bound load / store functors: per-unit state resolved once; loads are split into fetch (issue the global
// loads, keep the raw operands in registers) and make (combine them), so that a round's loads can be issued one
// round ahead of their use ---------------------------------------------------------------------------------------
// L2 eviction policy of the streams (work grids, tau, a(r) batches): evict_first keeps them from displacing the orbital planes
// that the next launches read again.  hint = 0 gives the normal policy (same instructions, for A/B runs).
__device__ __forceinline__ unsigned long long l2_policy(int hint) {
    unsigned long long p;
    if (hint) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    else asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void st_pol(cplx* p, cplx v, unsigned long long pol) {
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_pol(double* p, double v, unsigned long long pol) {
    asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(p), "d"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ cplx ld_pol(const cplx* p, unsigned long long pol) {
    cplx v;
    asm volatile("ld.global.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    return v;
}
// Work grids of the fused path are pruned (plan.h): element (x, column c) of packed grid b at b*gstride + x*ncols + c;
// cmap maps a plane offset y*NZ + z to c, or -1 where the spectrum is identically zero (not stored, read as 0).
struct LoadWorkC { const cplx* work; long gstride; const int* cmap; int ncols; int hint; };
struct StoreWorkC { cplx* work; long gstride; const int* cmap; int ncols; int hint; };
// Bound functors address one unit (packed grid b, plane x); `off` = y*NZ + z inside the plane.
struct BLoadWorkC {
    const cplx* g; const int* cmap; int ncols; unsigned long long pol;
    typedef cplx Raw;
    static constexpr int kModes = 1;
    __device__ __forceinline__ int mode() const { return 0; }
    template <int M> __device__ __forceinline__ Raw fetch(int off) const {
        const int c = __ldg(cmap + off);
        return c >= 0 ? ld_pol(g + c, pol) : make_double2(0.0, 0.0);
    }
    __device__ __forceinline__ Raw fetch_col(int c) const { return c >= 0 ? ld_pol(g + c, pol) : make_double2(0.0, 0.0); }
    __device__ __forceinline__ cplx make(const Raw& r) const { return r; }
    __device__ __forceinline__ void prefetch_l2(int, int tid, int nthr) const {      // the compact plane is one contiguous run
        for (int e = tid * 8; e < ncols; e += nthr * 8) asm volatile("prefetch.global.L2 [%0];" ::"l"(g + e));
    }
};
struct BStoreWorkC {
    cplx* g; const int* cmap; unsigned long long pol;
    __device__ __forceinline__ void operator()(int off, cplx v) const { const int c = __ldg(cmap + off); if (c >= 0) st_pol(g + c, v, pol); }
};
template <class L> struct HasColMap { static constexpr bool value = false; };      // loads that go through the pruned column map
template <> struct HasColMap<LoadWorkC> { static constexpr bool value = true; };
template <class S> struct StoresColMap { static constexpr bool value = false; };  // stores that go through the pruned column map
template <> struct StoresColMap<StoreWorkC> { static constexpr bool value = true; };
struct BLoadPair {
    const double *a0, *a1, *b0, *b1;   // re = a0*a1, im = imw*b0*b1 (imw = 0 for the odd last pair, which reuses a0, a1)
    double imw;
    struct Raw { double p, q, r, s; };
    static constexpr int kModes = 2;       // mode 1: b0 == a0 (consecutive pairs of one row share the first orbital): 3 loads
    __device__ __forceinline__ int mode() const { return b0 == a0 ? 1 : 0; }
    template <int M> __device__ __forceinline__ Raw fetch(int off) const {   // branch-free: the loads of a round issue back to back
        Raw w; w.p = __ldg(a0 + off); w.q = __ldg(a1 + off);
        w.r = (M == 1) ? w.p : __ldg(b0 + off);
        w.s = __ldg(b1 + off);
        return w;
    }
    __device__ __forceinline__ cplx make(const Raw& w) const { return make_double2(w.p * w.q, imw * (w.r * w.s)); }
    // pull the operand planes of the unit this CTA handles next into L2 (no registers held)
    __device__ __forceinline__ void prefetch_l2(int n, int tid, int nthr) const {
        for (int e = tid * 16; e < n; e += nthr * 16) {          // one 128-byte line = 16 doubles
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a0 + e));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a1 + e));
            if (b0 != a0) asm volatile("prefetch.global.L2 [%0];" ::"l"(b0 + e));
            if (b1 != a1) asm volatile("prefetch.global.L2 [%0];" ::"l"(b1 + e));
        }
    }
};
// Real-function batches (BatchLayout) addressed from one unit: both the chunked layout [nr/CHUNK][function][CHUNK] and the plain
// one [function][nr] (which is the chunked formula with a chunk stride of CHUNK elements) put point idx of function f at
//   f_off + (idx / CHUNK) * cstride + (idx % CHUNK),   f_off = f*CHUNK (chunked) or f*nr (plain).
// A bound functor keeps the byte address of (function, chunk of the plane's first point) and turns a plane offset into
// one shift, one mask and one 32x32->64 multiply-add.
struct UnitAddr {
    unsigned r0;        // (first point of the plane) & (CHUNK - 1)
    unsigned cs8;       // chunk stride in bytes
    __device__ __forceinline__ size_t operator()(int off) const {
        const unsigned i = r0 + (unsigned)off;
        return (size_t)(i >> CHUNK_LOG) * cs8 + (size_t)((i & (unsigned)(CHUNK - 1)) * 8u);
    }
};
__device__ __forceinline__ UnitAddr unit_addr(const BatchLayout& lay, long pbase) {
    return UnitAddr{(unsigned)(pbase & (CHUNK - 1)), (unsigned)((lay.chunked ? lay.cstride : CHUNK) * 8)};
}
__device__ __forceinline__ long fun_base(const BatchLayout& lay, long f, long pbase) {   // element offset of (f, chunk of pbase)
    return lay.chunked ? (pbase >> CHUNK_LOG) * lay.cstride + (lay.fbase + f) * CHUNK : (lay.fbase + f) * lay.nr + (pbase & ~(long)(CHUNK - 1));
}
struct BLoadPack2 {
    const char *p0, *q0; long d1; UnitAddr ua; bool has_im; double scale;   // p0/q0: function 2b of src0/src1 (q0 may be null); d1: bytes to 2b+1
    struct Raw { double p, q, r, s; };
    static constexpr int kModes = 1;
    __device__ __forceinline__ int mode() const { return 0; }
    template <int M> __device__ __forceinline__ Raw fetch(int off) const {
        const size_t o = ua(off);
        Raw w; w.p = *(const double*)(p0 + o); w.q = q0 ? *(const double*)(q0 + o) : 0.0; w.r = 0.0; w.s = 0.0;
        if (has_im) { w.r = *(const double*)(p0 + o + d1); if (q0) w.s = *(const double*)(q0 + o + d1); }
        return w;
    }
    __device__ __forceinline__ cplx make(const Raw& w) const { return make_double2((w.p + w.q) * scale, (w.r + w.s) * scale); }
    __device__ __forceinline__ void prefetch_l2(int, int, int) const {}
};
struct BStoreSplit2 {
    char* p0; long d1; UnitAddr ua; bool has_im; double scale; unsigned long long pol;
    __device__ __forceinline__ void operator()(int off, cplx v) const {
        char* q = p0 + ua(off);
        st_pol((double*)q, v.x * scale, pol);
        if (has_im) st_pol((double*)(q + d1), v.y * scale, pol);
    }
};
__device__ __forceinline__ BLoadWorkC bind(const LoadWorkC& l, int b, int x, long) { return BLoadWorkC{l.work + (long)b * l.gstride + (long)x * l.ncols, l.cmap, l.ncols, l2_policy(l.hint)}; }
__device__ __forceinline__ BStoreWorkC bind(const StoreWorkC& s, int b, int x, long) { return BStoreWorkC{s.work + (long)b * s.gstride + (long)x * s.ncols, s.cmap, l2_policy(s.hint)}; }
__device__ __forceinline__ BLoadPair bind(const LoadPair& l, int b, int, long pbase) {
    const int2 p0 = l.pairs[2 * b];
    BLoadPair r{l.phi + (long)p0.x * l.nr + pbase, l.phi2 + (long)p0.y * l.nr + pbase, nullptr, nullptr, 0.0};
    r.b0 = r.a0; r.b1 = r.a1;
    if (2 * b + 1 < l.npairs) { const int2 p1 = l.pairs[2 * b + 1]; r.b0 = l.phi + (long)p1.x * l.nr + pbase; r.b1 = l.phi2 + (long)p1.y * l.nr + pbase; r.imw = 1.0; }
    return r;
}
__device__ __forceinline__ BLoadPack2 bind(const LoadPack2& l, int b, int, long pbase) {
    const long e0 = fun_base(l.lay, 2L * b, pbase);
    return BLoadPack2{(const char*)(l.src0 + e0), l.src1 ? (const char*)(l.src1 + e0) : nullptr, l.lay.next() * 8, unit_addr(l.lay, pbase),
                      2 * b + 1 < l.nfun, l.scale};
}
__device__ __forceinline__ BStoreSplit2 bind(const StoreSplit2& s, int b, int, long pbase) {
    const bool has_im = 2 * b + 1 < s.nfun;
    long f0 = 2L * b, f1 = f0 + 1;
    if (s.slots) { f0 = s.slots[2 * b]; f1 = has_im ? s.slots[2 * b + 1] : f0; }
    return BStoreSplit2{(char*)(s.dst + fun_base(s.lay, f0, pbase)), (f1 - f0) * s.lay.next() * 8, unit_addr(s.lay, pbase), has_im, s.scale,
                        l2_policy(s.hint)};
}

// One phase = ITEMS butterflies spread over the CTA in rounds of NTHR.  The loads of round r+1 are issued before
// round r is computed and stored (double-buffered registers), so memory latency overlaps the butterflies.
// load(t, buf) fills buf for item t; work(t, buf) computes and stores item t.
template <int ITEMS, int NTHR, bool DB, class Buf, class LoadF, class WorkF>
__device__ __forceinline__ void run_rounds(int tid, LoadF&& load, WorkF&& work) {
    constexpr int NR = (ITEMS + NTHR - 1) / NTHR;
    if constexpr (DB) {
        Buf cur, nxt;
        if (tid < ITEMS) load(tid, cur);
#pragma unroll
        for (int r = 0; r < NR; ++r) {
            const int t = tid + r * NTHR;
            if (r + 1 < NR && t + NTHR < ITEMS) load(t + NTHR, nxt);
            if (t < ITEMS) work(t, cur);
            if (r + 1 < NR) cur = nxt;
        }
    } else {
        for (int t = tid; t < ITEMS; t += NTHR) { Buf cur; load(t, cur); work(t, cur); }
    }
}
template <class T, int R> struct RegBuf { T v[R]; };
// registers per thread that still let MINB CTAs of NTHR threads share the 64 K register file (warp granularity 8 regs)
template <int NTHR, int MINB> struct PlaneRegs {
    static constexpr int warps = ((NTHR + 31) / 32 + 3) / 4 * 4 * MINB;    // warps are allocated four at a time
    static constexpr int raw = 65536 / (warps * 32) / 8 * 8;
    static constexpr int value = raw > 255 ? 255 : raw;
};

// ---- plane kernel -------------------------------------------------------------------------------------------
// Persistent CTAs walk over the units (packed grid b, plane x) plane-major, unit u = x*batch + b: the CTAs running at the same
// time then work on the same few planes of all grids of the launch, and the orbital planes the pairs of a sub-block share
// are read from DRAM once and found in L2 (or L1) by the other pairs.  Flat index of (x, y, z) inside a grid: (x*NY + y)*NZ + z.
template <int NY, int NZ, int NTHR, int MINB, bool INV, bool DB1, bool DB2, class Load, class Store>
__global__ void __launch_bounds__(NTHR) __maxnreg__((PlaneRegs<NTHR, MINB>::value)) plane_kernel(Load ld, Store st, int nx, int nunits, int l2pf, const cplx* __restrict__ twy_g, const cplx* __restrict__ twz_g) {
    using TY = Two<NY>; using TZ = Two<NZ>;
    constexpr int R1y = TY::R1, R2y = TY::R2, R1z = TZ::R1, R2z = TZ::R2;
    constexpr int PITCH = TZ::PITCH;
    static_assert(NTHR % R2z == 0 && NTHR % R2y == 0, "a thread's residue must be the same in every round");
    extern __shared__ cplx sm[];
    const int tid = threadIdx.x;
    pdl_launch_dependents();
    cplx wz[R1z], wy[R1y];
    load_twiddles<R1z>(twz_g, tid % R2z, wz);
    if constexpr (NY == NZ) {
#pragma unroll
        for (int r = 0; r < R1y; ++r) wy[r] = wz[r];
    } else load_twiddles<R1y>(twy_g, tid % R2y, wy);
    typedef decltype(bind(ld, 0, 0, 0L)) BL;
    typedef typename BL::Raw Raw;
    const int nbatch = nunits / nx;
    constexpr int NR0 = (NZ * R1y + NTHR - 1) / NTHR;   // rounds of the first inverse stage
    int ccol[HasColMap<Load>::value ? NR0 : 1][R2y];
    if constexpr (HasColMap<Load>::value) {
#pragma unroll
        for (int r = 0; r < NR0; ++r) {
            const int t = tid + r * NTHR;
            const int k1 = t / NZ, zp = t - k1 * NZ;
#pragma unroll
            for (int i = 0; i < R2y; ++i) ccol[r][i] = (t < NZ * R1y) ? __ldg(ld.cmap + (k1 * R2y + i) * NZ + zp) : -1;
        }
    }
    // forward kernels storing to pruned work grids: the thread's 16-bit column indices of the last stage, two per register
    constexpr bool SCOLS = StoresColMap<Store>::value && !INV;
    static_assert(!SCOLS || NY * NZ < 65535, "16-bit column indices");
    unsigned scol[SCOLS ? NR0 : 1][(R2y + 1) / 2];
    if constexpr (SCOLS) {
#pragma unroll
        for (int r = 0; r < NR0; ++r) {
            const int t = tid + r * NTHR;
            const int k1 = t / NZ, zp = t - k1 * NZ;
#pragma unroll
            for (int h = 0; h < (R2y + 1) / 2; ++h) {
                unsigned pk = 0xffffffffu;
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int k = 2 * h + e;
                    int cc = -1;
                    if (k < R2y && t < NZ * R1y) cc = __ldg(st.cmap + (k1 * R2y + k) * NZ + zp);
                    const unsigned v = cc < 0 ? 0xffffu : (unsigned)cc;
                    pk = e == 0 ? ((pk & 0xffff0000u) | v) : ((pk & 0x0000ffffu) | (v << 16));
                }
                scol[r][h] = pk;
            }
        }
    }

    pdl_wait();
    for (int u = blockIdx.x; u < nunits; u += gridDim.x) {
        const int xpl = u / nbatch, b = u - xpl * nbatch;
        BL L = bind(ld, b, xpl, (long)xpl * NY * NZ);
        const auto S = bind(st, b, xpl, (long)xpl * NY * NZ);
        {   // operands of the unit this CTA takes next -> L2
            const int un = u + gridDim.x;
            if (l2pf && un < nunits) { const int xn = un / nbatch, bn = un - xn * nbatch; bind(ld, bn, xn, (long)xn * NY * NZ).prefetch_l2(NY * NZ, tid, NTHR); }
        }
        if constexpr (!INV) {
            // z stage 1 (radix R1z, twiddle after): global -> registers -> shared
            auto z1 = [&](auto mode_) {
                constexpr int MD = decltype(mode_)::value;
                run_rounds<NY * R2z, NTHR, DB1, RegBuf<Raw, R1z>>(tid,
                    [&](int t, RegBuf<Raw, R1z>& q) {
                        const int y = t / R2z, i = t - y * R2z;
#pragma unroll
                        for (int r = 0; r < R1z; ++r) q.v[r] = L.template fetch<MD>(y * NZ + i + R2z * r);
                    },
                    [&](int t, const RegBuf<Raw, R1z>& q) {
                        const int y = t / R2z, i = t - y * R2z;
                        cplx x[R1z];
#pragma unroll
                        for (int r = 0; r < R1z; ++r) x[r] = L.make(q.v[r]);
                        Dft<R1z, false>::run(x);
                        cplx* row = sm + y * PITCH;
                        row[TZ::pad(i)] = x[0];
#pragma unroll
                        for (int k = 1; k < R1z; ++k) row[TZ::pad(i + R2z * k)] = cmul(x[k], wz[k]);
                    });
            };
            if (BL::kModes > 1 && L.mode() == 1) z1(IC<1>{}); else z1(IC<0>{});
            __syncthreads();
            // z stage 2 (radix R2z on blocks of R2z consecutive positions), in place
            run_rounds<NY * R1z, NTHR, DB2, RegBuf<cplx, R2z>>(tid,
                [&](int t, RegBuf<cplx, R2z>& q) {
                    const int y = t / R1z, k1 = t - y * R1z;
                    const cplx* blk = sm + y * PITCH + TZ::pad(k1 * R2z);
#pragma unroll
                    for (int i = 0; i < R2z; ++i) q.v[i] = blk[i];
                },
                [&](int t, RegBuf<cplx, R2z>& q) {
                    const int y = t / R1z, k1 = t - y * R1z;
                    cplx* blk = sm + y * PITCH + TZ::pad(k1 * R2z);
                    Dft<R2z, false>::run(q.v);
#pragma unroll
                    for (int i = 0; i < R2z; ++i) blk[i] = q.v[i];
                });
            __syncthreads();
            // y stage 1 (radix R1y, twiddle after): lanes run over the residue i, the odd pitch keeps them on distinct banks
            run_rounds<NZ * R2y, NTHR, DB2, RegBuf<cplx, R1y>>(tid,
                [&](int t, RegBuf<cplx, R1y>& q) {
                    const int zp = t / R2y, i = t - zp * R2y;
                    const cplx* col = sm + TZ::pad(zp) + i * PITCH;
#pragma unroll
                    for (int r = 0; r < R1y; ++r) q.v[r] = col[r * R2y * PITCH];
                },
                [&](int t, RegBuf<cplx, R1y>& q) {
                    const int zp = t / R2y, i = t - zp * R2y;
                    cplx* col = sm + TZ::pad(zp) + i * PITCH;
                    Dft<R1y, false>::run(q.v);
                    col[0] = q.v[0];
#pragma unroll
                    for (int k = 1; k < R1y; ++k) col[k * R2y * PITCH] = cmul(q.v[k], wy[k]);
                });
            __syncthreads();
            // y stage 2 (radix R2y): shared -> registers -> global, lanes run over z (coalesced rows)
            if constexpr (SCOLS) {
#pragma unroll
                for (int r = 0; r < NR0; ++r) {
                    const int t = tid + r * NTHR;
                    if (t < NZ * R1y) {
                        const int k1 = t / NZ, zp = t - k1 * NZ;
                        const cplx* col = sm + TZ::pad(zp) + (k1 * R2y) * PITCH;
                        cplx x[R2y];
#pragma unroll
                        for (int i = 0; i < R2y; ++i) x[i] = col[i * PITCH];
                        Dft<R2y, false>::run(x);
#pragma unroll
                        for (int k = 0; k < R2y; ++k) {
                            const unsigned cc = (scol[r][k / 2] >> (16 * (k & 1))) & 0xffffu;
                            if (cc != 0xffffu) st_pol(S.g + cc, x[k], S.pol);
                        }
                    }
                }
            } else
            run_rounds<NZ * R1y, NTHR, DB2, RegBuf<cplx, R2y>>(tid,
                [&](int t, RegBuf<cplx, R2y>& q) {
                    const int k1 = t / NZ, zp = t - k1 * NZ;
                    const cplx* col = sm + TZ::pad(zp) + (k1 * R2y) * PITCH;
#pragma unroll
                    for (int i = 0; i < R2y; ++i) q.v[i] = col[i * PITCH];
                },
                [&](int t, RegBuf<cplx, R2y>& q) {
                    const int k1 = t / NZ, zp = t - k1 * NZ;
                    Dft<R2y, false>::run(q.v);
#pragma unroll
                    for (int k = 0; k < R2y; ++k) S((k1 * R2y + k) * NZ + zp, q.v[k]);
                });
        } else {
            // y inverse stage R2y: global -> registers -> shared
            if constexpr (HasColMap<Load>::value) {     // the thread's compact column indices are the same in every unit: registers
#pragma unroll
                for (int r = 0; r < NR0; ++r) {
                    const int t = tid + r * NTHR;
                    if (t < NZ * R1y) {
                        const int k1 = t / NZ, zp = t - k1 * NZ;
                        cplx x[R2y];
#pragma unroll
                        for (int i = 0; i < R2y; ++i) x[i] = L.fetch_col(ccol[r][i]);
                        Dft<R2y, true>::run(x);
                        cplx* col = sm + TZ::pad(zp) + (k1 * R2y) * PITCH;
#pragma unroll
                        for (int i = 0; i < R2y; ++i) col[i * PITCH] = x[i];
                    }
                }
            } else
            run_rounds<NZ * R1y, NTHR, DB1, RegBuf<Raw, R2y>>(tid,
                [&](int t, RegBuf<Raw, R2y>& q) {
                    const int k1 = t / NZ, zp = t - k1 * NZ;
#pragma unroll
                    for (int i = 0; i < R2y; ++i) q.v[i] = L.template fetch<0>((k1 * R2y + i) * NZ + zp);
                },
                [&](int t, const RegBuf<Raw, R2y>& q) {
                    const int k1 = t / NZ, zp = t - k1 * NZ;
                    cplx x[R2y];
#pragma unroll
                    for (int i = 0; i < R2y; ++i) x[i] = L.make(q.v[i]);
                    Dft<R2y, true>::run(x);
                    cplx* col = sm + TZ::pad(zp) + (k1 * R2y) * PITCH;
#pragma unroll
                    for (int i = 0; i < R2y; ++i) col[i * PITCH] = x[i];
                });
            __syncthreads();
            // y inverse stage R1y (conjugate twiddle before the butterfly), in place
            run_rounds<NZ * R2y, NTHR, DB2, RegBuf<cplx, R1y>>(tid,
                [&](int t, RegBuf<cplx, R1y>& q) {
                    const int zp = t / R2y, i = t - zp * R2y;
                    const cplx* col = sm + TZ::pad(zp) + i * PITCH;
#pragma unroll
                    for (int k = 0; k < R1y; ++k) q.v[k] = col[k * R2y * PITCH];
                },
                [&](int t, RegBuf<cplx, R1y>& q) {
                    const int zp = t / R2y, i = t - zp * R2y;
                    cplx* col = sm + TZ::pad(zp) + i * PITCH;
#pragma unroll
                    for (int k = 1; k < R1y; ++k) q.v[k] = cmulc(q.v[k], wy[k]);
                    Dft<R1y, true>::run(q.v);
#pragma unroll
                    for (int r = 0; r < R1y; ++r) col[r * R2y * PITCH] = q.v[r];
                });
            __syncthreads();
            // z inverse stage R2z, in place
            run_rounds<NY * R1z, NTHR, DB2, RegBuf<cplx, R2z>>(tid,
                [&](int t, RegBuf<cplx, R2z>& q) {
                    const int y = t / R1z, k1 = t - y * R1z;
                    const cplx* blk = sm + y * PITCH + TZ::pad(k1 * R2z);
#pragma unroll
                    for (int i = 0; i < R2z; ++i) q.v[i] = blk[i];
                },
                [&](int t, RegBuf<cplx, R2z>& q) {
                    const int y = t / R1z, k1 = t - y * R1z;
                    cplx* blk = sm + y * PITCH + TZ::pad(k1 * R2z);
                    Dft<R2z, true>::run(q.v);
#pragma unroll
                    for (int i = 0; i < R2z; ++i) blk[i] = q.v[i];
                });
            __syncthreads();
            // z inverse stage R1z: shared -> registers -> global (natural order)
            run_rounds<NY * R2z, NTHR, DB2, RegBuf<cplx, R1z>>(tid,
                [&](int t, RegBuf<cplx, R1z>& q) {
                    const int y = t / R2z, i = t - y * R2z;
                    const cplx* row = sm + y * PITCH;
#pragma unroll
                    for (int k = 0; k < R1z; ++k) q.v[k] = row[TZ::pad(i + R2z * k)];
                },
                [&](int t, RegBuf<cplx, R1z>& q) {
                    const int y = t / R2z, i = t - y * R2z;
#pragma unroll
                    for (int k = 1; k < R1z; ++k) q.v[k] = cmulc(q.v[k], wz[k]);
                    Dft<R1z, true>::run(q.v);
#pragma unroll
                    for (int r = 0; r < R1z; ++r) S(y * NZ + i + R2z * r, q.v[r]);
                });
        }
        __syncthreads();        // the plane buffer is reused by the next unit
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
    static constexpr int MINB = G > 12 ? 1 : (G > 9 ? 2 : 3);   // CTAs per SM the registers are budgeted for (radix-12 / radix-16 butterflies need more)
    static constexpr size_t SMEM = sizeof(cplx) * NX * XW;
};
// Twiddles: the residue / block index g = tid / XW is the warp index (XW = 32), so every stage dispatches on g to a
// body whose twiddles exp(-2 pi i g k / NX) are literals (mul_tw folds +-1, +-i and the octants): no twiddle registers
// or loads, 3 CTAs per SM.  The barriers stay outside the per-warp bodies.  (One generic body with warp-uniform twiddle loads
// is nine times less code and was measured in round 2: same speed within noise, 632.8 vs 630.6 ms of S4; not kept.)
template <int NX, int MODE>
__global__ void __launch_bounds__(XCfg<NX>::NTHR, XCfg<NX>::MINB) xpass_kernel(cplx* __restrict__ work, long inner, long nr, int batch,
                                                                 const cplx* __restrict__ tw_g, const double* __restrict__ ktab, int hint) {
    pdl_launch_dependents();
    const unsigned long long pol = l2_policy(hint);
    constexpr int R1 = XCfg<NX>::R1, R2 = XCfg<NX>::R2;
    extern __shared__ cplx sm[];
    const int tid = threadIdx.x, c = tid % XW, g = tid / XW;
    const long col = (long)blockIdx.x * XW + c;
    const bool live = col < inner;
    double kt[R2];
    if (MODE == SM_CONV) {
#pragma unroll
        for (int k = 0; k < R2; ++k) kt[k] = (live && g < R1) ? __ldg(ktab + (long)(g * R2 + k) * inner + col) : 0.0;
    }
    pdl_wait();
    for (int b = blockIdx.y; b < batch; b += gridDim.y) {
        cplx* gcol = work + (long)b * nr + col;
        if (MODE == SM_FWD || MODE == SM_CONV) {
            static_for<0, R2>([&](auto g_) {       // stage R1 forward of residue g: rows g + R2*r, twiddle after
                constexpr int GI = decltype(g_)::value;
                if (g == GI) {
                    cplx x[R1];
#pragma unroll
                    for (int r = 0; r < R1; ++r) x[r] = live ? ld_pol(gcol + (long)(GI + R2 * r) * inner, pol) : make_double2(0.0, 0.0);
                    Dft<R1, false>::run(x);
                    static_for<0, R1>([&](auto k_) {
                        constexpr int K = decltype(k_)::value;
                        sm[(GI + R2 * K) * XW + c] = mul_tw<false, NX, GI * K>(x[K]);
                    });
                }
            });
            __syncthreads();
        }
        if (g < R1) {           // block g: rows g*R2 + i
            cplx x[R2];
            if (MODE == SM_INV) {
#pragma unroll
                for (int i = 0; i < R2; ++i) x[i] = live ? ld_pol(gcol + (long)(g * R2 + i) * inner, pol) : make_double2(0.0, 0.0);
            } else {
#pragma unroll
                for (int i = 0; i < R2; ++i) x[i] = sm[(g * R2 + i) * XW + c];
                Dft<R2, false>::run(x);
            }
            if (MODE == SM_FWD) {
                if (live) {
#pragma unroll
                    for (int k = 0; k < R2; ++k) st_pol(gcol + (long)(g * R2 + k) * inner, x[k], pol);
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
            static_for<0, R2>([&](auto g_) {       // stage R1 inverse of residue g: conjugate twiddle, butterfly, natural order out
                constexpr int GI = decltype(g_)::value;
                if (g == GI) {
                    cplx x[R1];
                    static_for<0, R1>([&](auto k_) {
                        constexpr int K = decltype(k_)::value;
                        x[K] = mul_tw<true, NX, GI * K>(sm[(GI + R2 * K) * XW + c]);
                    });
                    Dft<R1, true>::run(x);
                    if (live) {
#pragma unroll
                        for (int r = 0; r < R1; ++r) st_pol(gcol + (long)(GI + R2 * r) * inner, x[r], pol);
                    }
                }
            });
        }
        __syncthreads();        // the tile is reused by the next grid of the batch
    }
}

// ---- x pass, generic body (long lengths) ----------------------------------------------------------------------------
// xpass_kernel gives every warp its own unrolled body with literal twiddles: 16 bodies for 128 = 16*8 are 6300 instructions (38 % of
// its stall samples wait for instruction fetch) and only the 8 residue warps of 16 work in the radix-16 stages.  Here every thread
// runs the same code over (butterfly, column) items, twiddles exp(-2 pi i g k / NX) from the table (L1 hits), XWG columns per CTA.
template <int NX> struct XGCfg {
    static constexpr int R1 = Two<NX>::R1, R2 = Two<NX>::R2;
    static constexpr int XWG = 32, NTHR = 256;
    static constexpr size_t SMEM = sizeof(cplx) * NX * XWG;
};
template <int NX, int MODE>
__global__ void __launch_bounds__(XGCfg<NX>::NTHR, 2) xpass_generic_kernel(cplx* __restrict__ work, long inner, long nr, int batch,
                                                                            const cplx* __restrict__ tw_g, const double* __restrict__ ktab, int hint) {
    pdl_launch_dependents();
    const unsigned long long pol = l2_policy(hint);
    constexpr int R1 = XGCfg<NX>::R1, R2 = XGCfg<NX>::R2, XWG = XGCfg<NX>::XWG, NTHR = XGCfg<NX>::NTHR;
    extern __shared__ cplx sm[];
    const int tid = threadIdx.x;
    pdl_wait();
    for (int b = blockIdx.y; b < batch; b += gridDim.y) {
        cplx* gbase = work + (long)b * nr + (long)blockIdx.x * XWG;
        if (MODE == SM_FWD || MODE == SM_CONV) {
            for (int t = tid; t < R2 * XWG; t += NTHR) {      // stage R1 forward of residue g: rows g + R2*r, twiddle after
                const int g = t / XWG, c = t - g * XWG;
                const bool live = (long)blockIdx.x * XWG + c < inner;
                cplx x[R1];
#pragma unroll
                for (int r = 0; r < R1; ++r) x[r] = live ? ld_pol(gbase + (long)(g + R2 * r) * inner + c, pol) : make_double2(0.0, 0.0);
                Dft<R1, false>::run(x);
                sm[g * XWG + c] = x[0];
#pragma unroll
                for (int k = 1; k < R1; ++k) sm[(g + R2 * k) * XWG + c] = cmul(x[k], __ldg(tw_g + g * k));
            }
            __syncthreads();
        }
        for (int t = tid; t < R1 * XWG; t += NTHR) {          // block g: rows g*R2 + i
            const int g = t / XWG, c = t - g * XWG;
            const long col = (long)blockIdx.x * XWG + c;
            const bool live = col < inner;
            cplx x[R2];
            if (MODE == SM_INV) {
#pragma unroll
                for (int i = 0; i < R2; ++i) x[i] = live ? ld_pol(gbase + (long)(g * R2 + i) * inner + c, pol) : make_double2(0.0, 0.0);
            } else {
#pragma unroll
                for (int i = 0; i < R2; ++i) x[i] = sm[(g * R2 + i) * XWG + c];
                Dft<R2, false>::run(x);
            }
            if (MODE == SM_FWD) {
                if (live) {
#pragma unroll
                    for (int k = 0; k < R2; ++k) st_pol(gbase + (long)(g * R2 + k) * inner + c, x[k], pol);
                }
            } else {
                if (MODE == SM_CONV) {
#pragma unroll
                    for (int k = 0; k < R2; ++k) { const double kt = live ? __ldg(ktab + (long)(g * R2 + k) * inner + col) : 0.0; x[k].x *= kt; x[k].y *= kt; }
                }
                Dft<R2, true>::run(x);
#pragma unroll
                for (int i = 0; i < R2; ++i) sm[(g * R2 + i) * XWG + c] = x[i];
            }
        }
        if (MODE != SM_FWD) {
            __syncthreads();
            for (int t = tid; t < R2 * XWG; t += NTHR) {      // stage R1 inverse of residue g: conjugate twiddle, butterfly, natural order out
                const int g = t / XWG, c = t - g * XWG;
                const bool live = (long)blockIdx.x * XWG + c < inner;
                cplx x[R1];
                x[0] = sm[g * XWG + c];
#pragma unroll
                for (int k = 1; k < R1; ++k) x[k] = cmulc(sm[(g + R2 * k) * XWG + c], __ldg(tw_g + g * k));
                Dft<R1, true>::run(x);
                if (live) {
#pragma unroll
                    for (int r = 0; r < R1; ++r) st_pol(gbase + (long)(g + R2 * r) * inner + c, x[r], pol);
                }
            }
        }
        __syncthreads();        // the tile is reused by the next grid of the batch
    }
}

}  // namespace tddft
