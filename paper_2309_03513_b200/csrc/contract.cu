// S5, the exchange contraction of Eq. 6:
//     out[(i0+i)*kc + k][r] -= alpha * sum_j tau_ij(r) a[(j0+j)*kc + k][r]          (and the transposed direction for i != j tiles)
// Per grid point this is a (ti x tj)(tj x kc) product whose matrices differ at every r: a batch of N_r small GEMMs on the FP64
// tensor pipe (mma.sync.m8n8k4.f64).  All real-space batches (tau, a, out) use the chunked layout [nr/CHUNK][function][CHUNK].
//
// CTA = 4 consecutive grid points (one 32-byte piece of every function's chunk) x the whole row block of the tile, 4 warps, two
// CTAs per SM.  Warp (pp, rh) owns the point pair pp (16 bytes of every row) and the row half rh (8*MT rows): its accumulators of
// out[I] (MT row tiles x 16 trial vectors x 2 points) and, for off-diagonal tiles, the DMMA B fragments of a[I] that the
// transposed product out[J] += tau^T a[I] needs stay in registers for the whole kernel (32*MT registers per lane).  The columns of
// the tile stream through a cp.async pipeline, 8 columns per stage (tau[IR rows][8 j] and a[8 j][16 k], 32-byte rows), NST stages,
// one CTA barrier per stage.  A tile may be any number of columns wide (api.cu makes the off-diagonal tiles as wide as the
// workspace allows): a[I] and out[I] cross HBM once per launch.
//
// Shared-memory layout.  Every fragment load is one LDS.128 that brings the values of BOTH points of the warp (two DMMAs per
// operand per load).  A quarter warp (8 lanes) reads 16 bytes from 8 different rows; the rows are 32 bytes, so the 16-byte piece
// p of row r is stored at  r*32 + ((p ^ ((r >> 2) & 1)) << 4)  and a quarter warp is conflict free iff its 8 rows are distinct
// mod 8.  tau element (i, jj) of a stage sits in row jj*IR + i with IR = 16*MT - 2 = 6 mod 8, so
//   direction 1 (A fragment, lane (lr, lc) -> i = 8m + lr, jj = 4s + lc):                rows lc*6 + lr         distinct mod 8
//   direction 2 (A fragment of tau^T, lane (lr, lc) -> jj = lr, i = 8(q/2) + 2(q%2) + (lc&1) + 4(lc/2)):  rows lr*6 + {0,1,4,5} (+2)
// (the contraction index of direction 2 is permuted inside blocks of 8 rows; the B fragments of a[I] use the same permutation),
// and a[j][k] of a stage sits in row (jj&3) | (k&1)<<2 | (k>>1)<<3 | (jj>>2)<<(3 + log2(KB/2)): rows lc + 4(lr&1) distinct mod 8.
// Every fragment load therefore costs the minimum of 4 wavefronts per 512 bytes (the round-1 kernel: one point per warp, LDS.64
// with an inherent two-way conflict, twice the wavefronts per DMMA: 48 % of the shared-memory pipe at 43 % of the DMMA pipe).
//
// The partial sums of direction 2 (two row halves) meet in shared memory (double buffered) and are subtracted from out[J] one
// stage later, behind the DMMAs of the next stage, in full 32-byte rows; the out[J] rows themselves are prefetched by cp.async two
// iterations ahead.  out[I] leaves through shared memory at the end.  Diagonal tiles (DIAG) read the packed upper triangle
// symmetrically and run direction 1 only: without the B fragments of a[I] (168 registers) and without the partial-sum and out[J]
// buffers (two stages = 64 KB) THREE of their CTAs fit an SM, three warps per scheduler instead of two.  No floating-point atomics:
// the summation order is fixed (reading A14).
//
// What bounds it (measured, profiles/r02_summary.md): with the DMMAs removed the kernel takes 0.78 of its time, with the stage
// copies removed 0.74: the CTA reads 32-byte pieces at a 256-byte stride (5.2 TB/s at best on this part, 7.4 TB/s for whole lines),
// and the prologue (a[I]) and epilogue (out[I]) of a CTA move a quarter of its bytes with nothing to overlap them.
#include "kernels.h"

namespace tddft {
namespace {

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
// 16-byte asynchronous copy; valid = false writes zeros (src-size 0) without touching global memory
__device__ __forceinline__ void cp16z(unsigned smem_addr, const void* gmem, bool valid) {
    const int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_addr), "l"(gmem), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ double2 lds128(unsigned addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts128(unsigned addr, double x, double y) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(x), "d"(y) : "memory");
}

constexpr int CP_P = 4;        // grid points per CTA
constexpr int CP_JS = 8;       // columns per stage
constexpr int CP_PF = 3;       // A fragments in flight ahead of the DMMAs
constexpr int CP_NTHR = 128;

// MT = row tiles of 8 per warp: a warp holds 8*MT rows, the CTA 16*MT; IR = rows per column of a stage = the largest row block.
// The per-warp state (accumulators + B fragments of a[I]) is 32*MT registers.  MT = 7 (tiles up to 110, 255 registers, two stages)
// leaves the compiler few registers to run fragment loads ahead of the DMMAs; MT = 6 (tiles up to 94, three stages) schedules
// better but needs 5 x 5 instead of 4 x 4 blocks at 432 orbitals: measured 319 ms against 305 ms for the whole S5 stage.
template <int NK, int MT> struct PipeCfg {
    static constexpr int HALF = 8 * MT;
    static constexpr int NST = MT >= 7 ? 2 : 3;             // stages in flight (what two CTAs per SM leave room for)
    static constexpr int IR = 16 * MT - 2;                  // = 6 mod 8 (fragment bank pattern above)
    static constexpr int KB = 8 * NK;                       // trial vectors per launch
    static constexpr int ASH = (NK == 2) ? 6 : 5;           // bit of (jj >> 2) in the row index of a[j][k]
    static constexpr int TROWS = CP_JS * IR;                // tau rows of a stage
    static constexpr int AROWS = CP_JS * KB;                // a[J] rows of a stage
    static constexpr int STAGE_B = (TROWS + AROWS) * 32;    // bytes
    static constexpr int FL_B = AROWS * 32;                 // one buffer of direction-2 partial sums (one row half) / of out[J] rows
    static constexpr size_t SMEM = (size_t)NST * STAGE_B + 4 * FL_B + 3 * FL_B;
    static constexpr size_t SMEM_DIAG = (size_t)2 * STAGE_B;        // diagonal tiles run direction 1 only: no partial-sum / out[J] buffers, two stages, three CTAs per SM
    static_assert(CHUNK % CP_P == 0 && IR % 8 == 6 && 2 * HALF >= IR, "fragment bank pattern / row coverage");
    static_assert(2 * HALF * KB * 32 <= 2 * STAGE_B, "prologue / epilogue stage the row block through the stage buffers");
};
__device__ __forceinline__ unsigned swz(int row, int piece) { return (unsigned)(row * 32 + ((piece ^ ((row >> 2) & 1)) << 4)); }

template <int NK, bool DIAG, int MT>
__global__ void __launch_bounds__(CP_NTHR, DIAG ? 3 : 2)
contract_pipe_kernel(double* __restrict__ out, const double* __restrict__ a, const double* __restrict__ tau,
                     int i0, int ti, int j0, int tj, int kc, int kn, long ftot, long stot, double alpha) {
    extern __shared__ __align__(128) char smc[];
    using C = PipeCfg<NK, MT>;
    constexpr int KB = C::KB, IR = C::IR, JS = CP_JS, NST = DIAG ? 2 : C::NST, HALF = C::HALF;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, lr = lane >> 2, lc = lane & 3;
    const int pp = w & 1, rh = w >> 1;
    const long chunk = blockIdx.x / (CHUNK / CP_P);
    const int pt0 = (int)(blockIdx.x % (CHUNK / CP_P)) * CP_P;
    const double* tau_c = tau + chunk * stot * CHUNK + pt0;
    const double* a_c = a + chunk * ftot * CHUNK + pt0;
    double* out_c = out + chunk * ftot * CHUNK + pt0;
    const unsigned sm0 = (unsigned)__cvta_generic_to_shared(smc);
    const unsigned fl0 = sm0 + NST * C::STAGE_B;            // [buffer][row half][AROWS][32 bytes]
    const unsigned oj0 = fl0 + 4 * C::FL_B;                 // out[J] rows of a stage, prefetched by cp.async: [stage % 3][AROWS][32 bytes]
    const int piece = tid & 1, rsub = tid >> 1;              // this thread's 16-byte piece of rows rsub, rsub + 64, ...

    // ---- prologue: a[I] -> shared memory (plain rows i*KB + k) -> B fragments of the transposed product
    double2 breg[DIAG ? 1 : 2 * MT][NK];
    if (!DIAG) {
        for (int row = rsub; row < 2 * HALF * KB; row += CP_NTHR / 2) {
            const int i = row / KB, kk = row - i * KB;
            const bool v = i < ti && kk < kn;
            cp16z(sm0 + row * 32 + piece * 16, v ? a_c + ((long)(i0 + i) * kc + kk) * CHUNK + piece * 2 : a_c, v);
        }
        cp_commit();
        cp_wait<0>();
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 2 * MT; ++q) {
            const int i = rh * HALF + 8 * (q >> 1) + 2 * (q & 1) + (lc & 1) + 4 * (lc >> 1);
#pragma unroll
            for (int n = 0; n < NK; ++n) breg[q][n] = lds128(sm0 + (i * KB + n * 8 + lr) * 32 + pp * 16);
        }
        __syncthreads();
    }

    // ---- stage loader: thread -> (column ljj, rows li0, li0 + 8, ..., piece lpc).  The tau slots of an off-diagonal tile are
    // column-major (slot = j*ti + i, api.cu: build_tiles) and a chunk is 4 points, so a column of the stage is ONE contiguous run
    // of ti*32 bytes and every copy address is the thread's base plus a literal (an LDGSTS reads its address registers late: a
    // loop that increments them waits on the long scoreboard).
    const int lpc = tid & 1, li0 = (tid >> 1) & 7, ljj = tid >> 4;
    const unsigned dst_t0 = swz(ljj * IR + li0, lpc);         // + 8 rows keeps the swizzle bit
    constexpr int NI = (IR + 7) / 8;
    auto load_stage = [&](int buf, int js) {
        const unsigned base = sm0 + buf * C::STAGE_B;
        const int col = js * JS + ljj;
        const bool cv = col < tj;
        const unsigned dst = base + dst_t0;
        if (DIAG) {
#pragma unroll
            for (int e = 0; e < NI; ++e) {
                const int i = li0 + 8 * e;
                if (i < IR) {
                    const bool v = cv && i < ti;
                    const int lo = min(i, col), hi = max(i, col);
                    cp16z(dst + e * 256, v ? tau_c + (long)(lo * (2 * tj - lo + 1) / 2 + (hi - lo)) * CHUNK + lpc * 2 : tau_c, v);     // slots fit 32 bits
                }
            }
        } else {
            const double* src = tau_c + ((long)(cv ? col : 0) * ti + li0) * CHUNK + lpc * 2;
            constexpr long sstep = 8L * CHUNK;
#pragma unroll
            for (int e = 0; e < NI; ++e) {
                const int i = li0 + 8 * e;
                if (i < IR) { const bool v = cv && i < ti; cp16z(dst + e * 256, v ? src + e * sstep : tau_c, v); }
            }
        }
#pragma unroll
        for (int e = 0; e < (C::AROWS + CP_NTHR / 2 - 1) / (CP_NTHR / 2); ++e) {
            const int rr = rsub + e * (CP_NTHR / 2);
            if (rr < C::AROWS) {
                const int jj = rr / KB, kk = rr - jj * KB, cj = js * JS + jj;
                const int ar = (jj & 3) | ((kk & 1) << 2) | ((kk >> 1) << 3) | ((jj >> 2) << C::ASH);
                const bool v = cj < tj && kk < kn;
                cp16z(base + C::TROWS * 32 + swz(ar, piece), v ? a_c + ((long)(j0 + cj) * kc + kk) * CHUNK + piece * 2 : a_c, v);
            }
        }
    };
    // rows of out[J] updated after the transposed product of stage js (one 32-byte row per thread): tid -> (jj, kk).  They are
    // fetched by cp.async two iterations before their use (with the copies of stage js+1), three buffers.
    const int fjj = tid / KB, fkk = tid - fjj * KB;
    auto flush_ptr = [&](int js) -> double* {
        const int col = js * JS + fjj;
        return (tid < C::AROWS && col < tj && fkk < kn) ? out_c + ((long)(j0 + col) * kc + fkk) * CHUNK : nullptr;
    };
    auto load_oj = [&](int js) {
        if (DIAG || js >= (tj + JS - 1) / JS) return;
        const double* p = flush_ptr(js);
        if (p) { const unsigned d = oj0 + (js % 3) * C::FL_B + tid * 32; cp16z(d, p, true); cp16z(d + 16, p + 2, true); }
    };
    auto flush_apply = [&](int js) {
        double* p = flush_ptr(js);
        if (!p) return;
        const unsigned f = fl0 + (js & 1) * 2 * C::FL_B + tid * 32, o = oj0 + (js % 3) * C::FL_B + tid * 32;
        const double2 d00 = lds128(f), d01 = lds128(f + 16), d10 = lds128(f + C::FL_B), d11 = lds128(f + C::FL_B + 16);
        const double2 o0 = lds128(o), o1 = lds128(o + 16);
        *(double2*)p = make_double2(fma(-alpha, d00.x + d10.x, o0.x), fma(-alpha, d00.y + d10.y, o0.y));
        *(double2*)(p + 2) = make_double2(fma(-alpha, d01.x + d11.x, o1.x), fma(-alpha, d01.y + d11.y, o1.y));
    };

    // ---- per-lane fragment addresses (byte offsets inside a stage)
    const unsigned offA1 = swz(lc * IR + rh * HALF + lr, pp);                             // + m*256 + s*4*IR*32
    const unsigned offB1 = C::TROWS * 32 + swz(lc + 4 * (lr & 1) + 8 * (lr >> 1), pp);    // + n*32*32 + s*4*KB*32
    const unsigned offA2e = swz(lr * IR + rh * HALF + (lc & 1) + 4 * (lc >> 1), pp);      // + (q>>1)*256
    const unsigned offA2o = swz(lr * IR + rh * HALF + 2 + (lc & 1) + 4 * (lc >> 1), pp);

    double acc[MT][NK][2][2];            // [row tile][k half][point][fragment element]
#pragma unroll
    for (int m = 0; m < MT; ++m)
#pragma unroll
        for (int n = 0; n < NK; ++n) { acc[m][n][0][0] = 0.0; acc[m][n][0][1] = 0.0; acc[m][n][1][0] = 0.0; acc[m][n][1][1] = 0.0; }

    const int nst = (tj + JS - 1) / JS;
#pragma unroll
    for (int st = 0; st < NST - 1; ++st) {
        if (st < nst) load_stage(st, st);
        if (st == NST - 2) load_oj(0);
        cp_commit();
    }
    for (int js = 0; js < nst; ++js) {
        cp_wait<NST - 2>();
        __syncthreads();                 // stage js has landed for everyone; stage js-1 is consumed and its partial sums are written
        if (js + NST - 1 < nst) load_stage((js + NST - 1) % NST, js + NST - 1);
        load_oj(js + 1);
        cp_commit();
        const unsigned S = sm0 + (js % NST) * C::STAGE_B;
        // direction 1: out[i][k] += sum_j tau[i][j] a[j][k]
#pragma unroll
        for (int s = 0; s < JS / 4; ++s) {
            double2 bf[NK];
#pragma unroll
            for (int n = 0; n < NK; ++n) bf[n] = lds128(S + offB1 + n * 32 * 32 + s * 4 * KB * 32);
            const unsigned Ap = S + offA1 + s * 4 * IR * 32;
            double2 afq[CP_PF];
#pragma unroll
            for (int m = 0; m < CP_PF; ++m) afq[m] = lds128(Ap + m * 256);
#pragma unroll
            for (int m = 0; m < MT; ++m) {
                const double2 af = afq[m % CP_PF];
                if (m + CP_PF < MT) afq[m % CP_PF] = lds128(Ap + (m + CP_PF) * 256);
#pragma unroll
                for (int n = 0; n < NK; ++n) {
                    dmma884(acc[m][n][0][0], acc[m][n][0][1], af.x, bf[n].x);
                    dmma884(acc[m][n][1][0], acc[m][n][1][1], af.y, bf[n].y);
                }
            }
        }
        if (!DIAG) {
            if (js > 0) flush_apply(js - 1);
            // direction 2: out[j][k] += sum_i tau[i][j] a[i][k], the 8 columns of this stage, this warp's row half
            double acc2[NK][2][2];
#pragma unroll
            for (int n = 0; n < NK; ++n) { acc2[n][0][0] = 0.0; acc2[n][0][1] = 0.0; acc2[n][1][0] = 0.0; acc2[n][1][1] = 0.0; }
            double2 atq[CP_PF];
#pragma unroll
            for (int q = 0; q < CP_PF; ++q) atq[q] = lds128(S + ((q & 1) ? offA2o : offA2e) + (q >> 1) * 256);
#pragma unroll
            for (int q = 0; q < 2 * MT; ++q) {
                const double2 af = atq[q % CP_PF];
                if (q + CP_PF < 2 * MT) atq[q % CP_PF] = lds128(S + (((q + CP_PF) & 1) ? offA2o : offA2e) + ((q + CP_PF) >> 1) * 256);
#pragma unroll
                for (int n = 0; n < NK; ++n) {
                    dmma884(acc2[n][0][0], acc2[n][0][1], af.x, breg[q][n].x);
                    dmma884(acc2[n][1][0], acc2[n][1][1], af.y, breg[q][n].y);
                }
            }
            // C fragment: lane holds (row lr = column jj of the stage, trial vectors n*8 + 2 lc, + 1) for both points
            const unsigned f = fl0 + ((js & 1) * 2 + rh) * C::FL_B + pp * 16;
#pragma unroll
            for (int n = 0; n < NK; ++n) {
                sts128(f + (lr * KB + n * 8 + 2 * lc) * 32, acc2[n][0][0], acc2[n][1][0]);
                sts128(f + (lr * KB + n * 8 + 2 * lc + 1) * 32, acc2[n][0][1], acc2[n][1][1]);
            }
        }
    }
    cp_wait<0>();
    __syncthreads();
    if (!DIAG) flush_apply(nst - 1);      // partial sums of the last stage
    // ---- epilogue: out[I] -= alpha * acc through shared memory (full rows; plain rows i*KB + k)
#pragma unroll
    for (int m = 0; m < MT; ++m)
#pragma unroll
        for (int n = 0; n < NK; ++n) {
            const unsigned r = sm0 + (((rh * HALF + m * 8 + lr) * KB + n * 8 + 2 * lc) * 32) + pp * 16;
            sts128(r, acc[m][n][0][0], acc[m][n][1][0]);
            sts128(r + 32, acc[m][n][0][1], acc[m][n][1][1]);
        }
    __syncthreads();
    constexpr int EB = 8;                // rows in flight per thread: the loads of a batch are issued before its stores
    for (int row0 = rsub; row0 < ti * KB; row0 += EB * (CP_NTHR / 2)) {
        double2 o[EB]; double* p[EB];
#pragma unroll
        for (int e = 0; e < EB; ++e) {
            const int row = row0 + e * (CP_NTHR / 2), i = row / KB, kk = row - i * KB;
            p[e] = (row < ti * KB && kk < kn) ? out_c + ((long)(i0 + i) * kc + kk) * CHUNK + piece * 2 : nullptr;
            o[e] = p[e] ? *(const double2*)p[e] : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int e = 0; e < EB; ++e) {
            if (p[e]) {
                const double2 d = lds128(sm0 + (row0 + e * (CP_NTHR / 2)) * 32 + piece * 16);
                *(double2*)p[e] = make_double2(fma(-alpha, d.x, o[e].x), fma(-alpha, d.y, o[e].y));
            }
        }
    }
}

template <int NK, bool DIAG, int MT>
cudaError_t pipe_launch(long nchunks, double* out, const double* a, const double* tau, int i0, int ti, int j0, int tj,
                        int kc, int kn, long ftot, long stot, double alpha, cudaStream_t st) {
    constexpr size_t smem = DIAG ? PipeCfg<NK, MT>::SMEM_DIAG : PipeCfg<NK, MT>::SMEM;
    static bool attr_done[kMaxDevices] = {false};
    const int dev = current_device();
    if (!attr_done[dev]) {
        cudaError_t e = cudaFuncSetAttribute(contract_pipe_kernel<NK, DIAG, MT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_done[dev] = true;
    }
    contract_pipe_kernel<NK, DIAG, MT><<<(unsigned)(nchunks * (CHUNK / CP_P)), CP_NTHR, smem, st>>>(out, a, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha);
    return cudaGetLastError();
}
template <int MT>
cudaError_t pipe_shape(bool diag, long nchunks, double* o, const double* ap, const double* tau, int i0, int ti, int j0, int tj,
                       int kc, int kn, long ftot, long stot, double alpha, cudaStream_t st) {
    if (kn > 8) return diag ? pipe_launch<2, true, MT>(nchunks, o, ap, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha, st)
                            : pipe_launch<2, false, MT>(nchunks, o, ap, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha, st);
    return diag ? pipe_launch<1, true, MT>(nchunks, o, ap, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha, st)
                : pipe_launch<1, false, MT>(nchunks, o, ap, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha, st);
}

constexpr int kTileSmall = PipeCfg<2, 4>::IR, kTilePref = PipeCfg<2, 6>::IR, kTileMax = PipeCfg<2, 7>::IR;

}  // namespace

int contract_full_max_tile() { return kTileMax; }
int contract_full_pref_tile() { return kTileMax; }
cudaError_t launch_contract_full(bool diag, double* out, const double* a, const double* tau, int i0, int ti, int j0, int tj, int kc,
                                 long ftot, long stot, long nr, double alpha, cudaStream_t st) {
    if (ti > kTileMax || tj < 1 || ti < 1 || (diag && ti != tj)) return cudaErrorInvalidValue;
    const long nchunks = (nr + CHUNK - 1) / CHUNK;
    for (int kb = 0; kb < kc; kb += 16) {
        const int kn = kc - kb < 16 ? kc - kb : 16;
        double* o = out + (long)kb * CHUNK; const double* ap = a + (long)kb * CHUNK;
        cudaError_t e = ti <= kTileSmall ? pipe_shape<4>(diag, nchunks, o, ap, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha, st)
                      : ti <= kTilePref  ? pipe_shape<6>(diag, nchunks, o, ap, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha, st)
                                         : pipe_shape<7>(diag, nchunks, o, ap, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha, st);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace tddft
