// Pointwise, scatter/gather, contraction and LDA kernels of the Liouville hot path (hand-written CUDA, sm_100a).
#include <algorithm>
#include "kernels.h"

namespace tddft {

// ------------------------------------------------------------------------------------------------------
__global__ void scatter_pack2_kernel(const cplx* __restrict__ X, FunLayout lay, int f0, int nfun,
                                     const int* __restrict__ idx_p, const int* __restrict__ idx_m,
                                     cplx* __restrict__ work, long nr) {
    const int b = blockIdx.y;
    const int fa = f0 + 2 * b, fb = fa + 1;
    const cplx* xa = X + (long)(lay.k0 + fa % lay.kc) * lay.vec_len + lay.block_off + (long)(fa / lay.kc) * lay.npwh;
    const cplx* xb = (fb < nfun) ? X + (long)(lay.k0 + fb % lay.kc) * lay.vec_len + lay.block_off + (long)(fb / lay.kc) * lay.npwh : nullptr;
    cplx* w = work + (long)b * nr;
    for (long g = blockIdx.x * (long)blockDim.x + threadIdx.x; g < lay.npwh; g += (long)gridDim.x * blockDim.x) {
        cplx za = xa[g];
        cplx zb = xb ? xb[g] : make_double2(0.0, 0.0);
        if (g == 0) { w[idx_p[0]] = make_double2(za.x, zb.x); continue; }   // Im c(0) = 0 by convention
        w[idx_p[g]] = make_double2(za.x - zb.y, za.y + zb.x);   // za + i zb
        w[idx_m[g]] = make_double2(za.x + zb.y, zb.x - za.y);   // conj(za) + i conj(zb)
    }
}
cudaError_t launch_scatter_pack2(const cplx* X, FunLayout lay, int f0, int nfun, int batch, const int* idx_p, const int* idx_m,
                                 cplx* work, long nr, cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(work, 0, sizeof(cplx) * nr * batch, st);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)((lay.npwh + 255) / 256), (unsigned)batch);
    scatter_pack2_kernel<<<grid, 256, 0, st>>>(X, lay, f0, nfun, idx_p, idx_m, work, nr);
    return cudaGetLastError();
}

__global__ void gather_unpack2_kernel(const cplx* __restrict__ work, long nr, const int* __restrict__ idx_p,
                                      const int* __restrict__ idx_m, int f0, int nfun, double scale,
                                      const cplx* __restrict__ X, cplx* __restrict__ AX, FunLayout lay,
                                      const double* __restrict__ kin, const double* __restrict__ eig) {
    const int b = blockIdx.y;
    const int fa = f0 + 2 * b, fb = fa + 1;
    const int va = fa / lay.kc, vb = fb / lay.kc;
    const long oa = (long)(lay.k0 + fa % lay.kc) * lay.vec_len + lay.block_off + (long)va * lay.npwh;
    const long ob = (long)(lay.k0 + fb % lay.kc) * lay.vec_len + lay.block_off + (long)vb * lay.npwh;
    const bool hb = fb < nfun;
    const double ea = X ? eig[va] : 0.0, eb = (X && hb) ? eig[vb] : 0.0;
    const cplx* w = work + (long)b * nr;
    for (long g = blockIdx.x * (long)blockDim.x + threadIdx.x; g < lay.npwh; g += (long)gridDim.x * blockDim.x) {
        const cplx zp = w[idx_p[g]], zm = w[idx_m[g]];
        // c_A = (Z(G) + conj Z(-G))/2,  c_B = (Z(G) - conj Z(-G))/(2i)
        if (!X) {      // plain transform to the sphere, no D term
            AX[oa + g] = make_double2(0.5 * scale * (zp.x + zm.x), 0.5 * scale * (zp.y - zm.y));
            if (hb) AX[ob + g] = make_double2(0.5 * scale * (zp.y + zm.y), -0.5 * scale * (zp.x - zm.x));
            continue;
        }
        const double k = kin[g];
        cplx xa = X[oa + g];
        AX[oa + g] = make_double2(fma(0.5 * scale, zp.x + zm.x, (k - ea) * xa.x), fma(0.5 * scale, zp.y - zm.y, (k - ea) * xa.y));
        if (hb) {
            cplx xb = X[ob + g];
            AX[ob + g] = make_double2(fma(0.5 * scale, zp.y + zm.y, (k - eb) * xb.x), fma(-0.5 * scale, zp.x - zm.x, (k - eb) * xb.y));
        }
    }
}
cudaError_t launch_gather_unpack2(const cplx* work, long nr, const int* idx_p, const int* idx_m, int f0, int nfun, int batch,
                                  double scale, const cplx* X, cplx* AX, FunLayout lay, const double* kin, const double* eig,
                                  cudaStream_t st) {
    dim3 grid((unsigned)((lay.npwh + 255) / 256), (unsigned)batch);
    gather_unpack2_kernel<<<grid, 256, 0, st>>>(work, nr, idx_p, idx_m, f0, nfun, scale, X, AX, lay, kin, eig);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------
// a is in the chunked layout [nr/32][nocc*kc][32] (common.h); phi and drho are plain [.][nr]
template <int KC>
__global__ void drho_kernel(const double* __restrict__ phi, const double* __restrict__ a, int nocc, int kc, int kk0, long nr,
                            double* __restrict__ drho) {
    const long r = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (r >= nr) return;
    double acc[KC];
#pragma unroll
    for (int q = 0; q < KC; ++q) acc[q] = 0.0;
    const double* ac = a + (r >> 5) * ((long)nocc * kc * CHUNK) + (r & (CHUNK - 1));
    for (int v = 0; v < nocc; ++v) {
        const double p = phi[(long)v * nr + r];
        const double* av = ac + ((long)v * kc + kk0) * CHUNK;
#pragma unroll
        for (int q = 0; q < KC; ++q) if (kk0 + q < kc) acc[q] = fma(p, av[q * CHUNK], acc[q]);
    }
#pragma unroll
    for (int q = 0; q < KC; ++q) if (kk0 + q < kc) drho[(long)(kk0 + q) * nr + r] = acc[q];
}
cudaError_t launch_drho(const double* phi, const double* a, int nocc, int kc, long nr, double* drho, cudaStream_t st) {
    const unsigned nb = (unsigned)((nr + 127) / 128);
    for (int kk0 = 0; kk0 < kc; kk0 += 4) drho_kernel<4><<<nb, 128, 0, st>>>(phi, a, nocc, kc, kk0, nr, drho);
    return cudaGetLastError();
}

__global__ void hxc_potential_kernel(const double* __restrict__ vh, const double* __restrict__ f0, const double* __restrict__ d0,
                                     const double* __restrict__ f1, const double* __restrict__ d1, long nr, double* __restrict__ V) {
    const long r = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (r >= nr) return;
    const long o = (long)blockIdx.y * nr + r;
    double v = vh[o] + f0[r] * d0[o];
    if (f1) v += f1[r] * d1[o];
    V[o] = v;
}
cudaError_t launch_hxc_potential(const double* vh, const double* f0, const double* drho0, const double* f1, const double* drho1,
                                 int kc, long nr, double* V, cudaStream_t st) {
    dim3 grid((unsigned)((nr + 255) / 256), (unsigned)kc);
    hxc_potential_kernel<<<grid, 256, 0, st>>>(vh, f0, drho0, f1, drho1, nr, V);
    return cudaGetLastError();
}

// One CTA = one chunk of 32 grid points, all functions: the chunk's nocc*kc rows of 256 bytes are one contiguous run of `out`.
__global__ void out_init_kernel(const double* __restrict__ phi, const double* __restrict__ V, const double* __restrict__ vloc,
                                const double* __restrict__ a, int nocc, int kc, long nr, double* __restrict__ out) {
    const long chunk = blockIdx.x;
    const int lane = threadIdx.x & (CHUNK - 1), sub = threadIdx.x / CHUNK, nsub = blockDim.x / CHUNK;
    const long r = chunk * CHUNK + lane;
    const bool live = r < nr;
    const long base = chunk * ((long)nocc * kc * CHUNK) + lane;
    const double vl = (vloc && live) ? vloc[r] : 0.0;
    for (int v = sub; v < nocc; v += nsub) {
        const double p = (V && live) ? phi[(long)v * nr + r] : 0.0;
        for (int kk = 0; kk < kc; ++kk) {
            const long o = base + ((long)v * kc + kk) * CHUNK;
            double y = 0.0;
            if (live) {
                if (V) y = p * __ldg(V + (long)kk * nr + r);
                if (vloc) y = fma(vl, a[o], y);
            }
            out[o] = y;
        }
    }
}
cudaError_t launch_out_init(const double* phi, const double* V, const double* vloc, const double* a, int nocc, int kc, long nr,
                            double* out, cudaStream_t st) {
    const long nchunks = (nr + CHUNK - 1) / CHUNK;
    if (!V && !vloc) return cudaMemsetAsync(out, 0, sizeof(double) * nchunks * CHUNK * nocc * kc, st);
    out_init_kernel<<<(unsigned)nchunks, 256, 0, st>>>(phi, V, vloc, a, nocc, kc, nr, out);
    return cudaGetLastError();
}

// S5: out[(i0+i)*kc+k][r] -= alpha * sum_j tau_ij(r) a[(j0+j)*kc+k][r]   (Eq. 6).
// Per grid point this is a (ti x tj)(tj x kc) product whose matrices differ at every r: a batch of N_r small GEMMs,
// run on the FP64 tensor pipe (mma.sync.m8n8k4.f64).  All real-space batches (tau, a, out) use the chunked layout
// [nr/32][function][32].
__device__ __forceinline__ void dmma884k(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ------------------------------------------------------------------------------------------------------
// S5, register-resident tiles.  One warp owns ONE grid point and keeps the whole row block of the tile in registers:
// the accumulators of out[I] (up to 112 rows x 16 trial vectors = 56 doubles per lane) and, for off-diagonal tiles,
// the B fragments of a[I] (54 doubles) that the transposed product out[J] += tau^T a[I] needs.  The CTA (FT_P = 4 warps =
// 4 consecutive points, two CTAs per SM) sweeps the columns of the tile 8 at a time through a double-buffered cp.async
// stage (tau[all i][8 j] and a[8 j][16 k], 32-byte rows padded to 48 bytes); every tau element is loaded into the SM once
// and used for both directions: 110 DMMAs per warp between barriers and ~0.14 bytes of L2->SM traffic per flop instead
// of 0.375.  Row pitch FT_PITCH = 6 doubles and 108 rows per column make (row stride) = 8 mod 16 doubles, so both
// fragment patterns (lanes over (i, j) for tau and over (j, i) for tau^T) spread over 8 distinct 8-byte banks: 4
// wavefronts per load.  (Measured and rejected in round 2: storing tau with the two points of a 16-byte piece swapped in
// alternate rows so that a half warp hits 16 different banks -- 2 wavefronts per load -- made the kernel 5 % slower, 352 vs
// 333 ms: shared-memory wavefronts are not what limits it.)  Results leave through shared memory so that every global access
// is a full 32-byte row.
// Tile shapes: MT row tiles of 8 per warp, IR rows per column in a stage (= largest row block; IR = 4 mod 8 for the bank pattern).
// The smaller shape leaves registers for the compiler to run fragment loads ahead of the DMMAs.
struct FullShapeL { static constexpr int MT = 14, IR = 108; static constexpr int TMAX = 108; };
struct FullShapeS { static constexpr int MT = 11, IR = 92; static constexpr int TMAX = 88; };
constexpr int FT_P = 4;          // grid points (= warps) per CTA: two CTAs per SM, so one CTA's prologue/epilogue hides behind the other's DMMAs
constexpr int FT_PPR = FT_P / 2; // 16-byte pieces per shared-memory row
constexpr int FT_PITCH = FT_P + 2;   // doubles per shared-memory row (rows stay 16-byte aligned)
constexpr int FT_JS = 8;         // columns per stage
constexpr int FT_PF = 3;         // A fragments in flight ahead of the DMMAs (5 measured no better, copies interleaved with the DMMAs worse)
template <int NK, class SH> struct FullCfg {
    static constexpr int FT_MT = SH::MT, FT_IR = SH::IR;
    static_assert((FT_IR * FT_PITCH) % 16 == 8 && FT_PITCH % 2 == 0 && FT_IR >= SH::TMAX, "fragment bank pattern");
    static constexpr int KB = 8 * NK;                                   // trial vectors per launch
    static constexpr int ROWS = FT_JS * FT_IR + FT_JS * KB;             // rows of one stage
    static constexpr int STAGE = ROWS * FT_PITCH;                       // doubles
    static constexpr int FLUSH = FT_JS * KB * FT_PITCH;                 // doubles (two of them: products and prefetched out[J] rows)
    static constexpr size_t SMEM = sizeof(double) * (2 * STAGE + 2 * FLUSH);
    static_assert(FT_MT * 8 * KB * FT_PITCH <= 2 * STAGE, "the epilogue stages the row block through the two stage buffers");
};
template <int NK, bool DIAG, class SH>
__global__ void __launch_bounds__(32 * FT_P, 2)
contract_full_kernel(double* __restrict__ out, const double* __restrict__ a, const double* __restrict__ tau,
                     int i0, int ti, int j0, int tj, int kc, int kn, long ftot, long stot, double alpha) {
    extern __shared__ __align__(16) double sm[];
    using C = FullCfg<NK, SH>;
    constexpr int FT_MT = SH::MT, FT_IR = SH::IR;
    constexpr int KB = C::KB, IR = FT_IR, PITCH = FT_PITCH, JS = FT_JS, PPR = FT_PPR;
    constexpr int NTHR = 32 * FT_P, RSTEP = NTHR / PPR;     // rows covered by one pass of the CTA over 16-byte pieces
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, lr = lane >> 2, lc = lane & 3;
    const long chunk = blockIdx.x / (CHUNK / FT_P);
    const int pt0 = (int)(blockIdx.x % (CHUNK / FT_P)) * FT_P;
    const double* tau_c = tau + chunk * stot * CHUNK + pt0;
    const double* a_c = a + chunk * ftot * CHUNK + pt0;
    double* out_c = out + chunk * ftot * CHUNK + pt0;
    const int piece2 = (tid % PPR) * 2, rsub = tid / PPR;    // this thread's 16-byte piece of rows rsub, rsub + RSTEP, ...
    double* fl = sm + 2 * C::STAGE;                          // products of the transposed direction, [8 j * KB][PITCH]
    double* ojs = fl + C::FLUSH;                             // the out[J] rows they are subtracted from, prefetched by cp.async

    // ---- prologue: a[I] -> shared memory (coalesced) -> B fragments of the transposed product
    double breg[DIAG ? 1 : IR / 4][NK];
    if (!DIAG) {
        for (int row = rsub; row < IR * KB; row += RSTEP) {
            const int i = row / KB, kk = row - i * KB;
            double* dst = sm + row * PITCH + piece2;
            if (i < ti && kk < kn) cp_async16(dst, a_c + ((long)(i0 + i) * kc + kk) * CHUNK + piece2);
            else *(double2*)dst = make_double2(0.0, 0.0);
        }
        cp_async_commit();
        cp_async_wait<0>();
        __syncthreads();
#pragma unroll
        for (int q = 0; q < IR / 4; ++q)
#pragma unroll
            for (int n = 0; n < NK; ++n) breg[q][n] = sm[((q * 4 + lc) * KB + n * 8 + lr) * PITCH + w];
        __syncthreads();
    }
    // Stage loader.  tau part: a group of 8*PPR lanes copies the pieces of the 8 columns of one row i; rows advance by a
    // constant, so a copy costs a pointer increment.  a part: 8*KB rows spread over the CTA.
    constexpr int LPR = 8 * PPR, RPW = 32 / LPR, ISTEP = FT_P * RPW;
    const int ljj = (lane % LPR) / PPR, lp2 = (lane % PPR) * 2, li0 = w * RPW + lane / LPR;
    auto load_stage = [&](int buf, int js) {
        double* base = sm + buf * C::STAGE;
        const int col = js * JS + ljj;
        double* dst = base + (ljj * IR + li0) * PITCH + lp2;
        if (col < tj) {
            if (DIAG) {
#pragma unroll 2
                for (int i = li0; i < IR; i += ISTEP, dst += ISTEP * PITCH) {
                    if (i < ti) {
                        const int lo = min(i, col), hi = max(i, col);
                        cp_async16(dst, tau_c + (long)(lo * (2 * tj - lo + 1) / 2 + (hi - lo)) * CHUNK + lp2);     // slots fit 32 bits
                    } else *(double2*)dst = make_double2(0.0, 0.0);
                }
            } else {
                const double* src = tau_c + ((long)li0 * tj + col) * CHUNK + lp2;
                const long sstep = (long)ISTEP * tj * CHUNK;
#pragma unroll 2
                for (int i = li0; i < IR; i += ISTEP, dst += ISTEP * PITCH, src += sstep) {
                    if (i < ti) cp_async16(dst, src);
                    else *(double2*)dst = make_double2(0.0, 0.0);
                }
            }
        } else {
            for (int i = li0; i < IR; i += ISTEP, dst += ISTEP * PITCH) *(double2*)dst = make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int e = 0; e < (JS * KB + RSTEP - 1) / RSTEP; ++e) {
            const int rr = rsub + e * RSTEP;
            if (rr < JS * KB) {
                const int jj = rr / KB, kk = rr - jj * KB, cj = js * JS + jj;
                double* d2 = base + (JS * IR + rr) * PITCH + piece2;
                if (cj < tj && kk < kn) cp_async16(d2, a_c + ((long)(j0 + cj) * kc + kk) * CHUNK + piece2);
                else *(double2*)d2 = make_double2(0.0, 0.0);
            }
        }
    };
    constexpr int NFL = (JS * KB + RSTEP - 1) / RSTEP;      // rows of out[J] per thread and stage
    double acc[FT_MT][NK][2];
#pragma unroll
    for (int m = 0; m < FT_MT; ++m)
#pragma unroll
        for (int n = 0; n < NK; ++n) { acc[m][n][0] = 0.0; acc[m][n][1] = 0.0; }
    const int nst = (tj + JS - 1) / JS;
    load_stage(0, 0);
    cp_async_commit();
    for (int js = 0; js < nst; ++js) {
        cp_async_wait<0>();
        __syncthreads();                 // stage js has landed for everyone; stage js-1 and its flush are consumed
        if (!DIAG) {                     // rows of out[J] this thread updates after the transposed product: fetched behind the DMMAs
#pragma unroll
            for (int e = 0; e < NFL; ++e) {
                const int row = rsub + e * RSTEP, jj = row / KB, kk = row - jj * KB, col = js * JS + jj;
                if (row < JS * KB && col < tj && kk < kn) cp_async16(ojs + row * PITCH + piece2, out_c + ((long)(j0 + col) * kc + kk) * CHUNK + piece2);
            }
        }
        cp_async_commit();
        if (js + 1 < nst) load_stage((js + 1) & 1, js + 1);
        cp_async_commit();
        const double* S = sm + (js & 1) * C::STAGE + w;
        // direction 1: out[i][k] += sum_j tau[i][j] a[j][k]
#pragma unroll
        for (int s = 0; s < JS / 4; ++s) {
            double bf[NK];
#pragma unroll
            for (int n = 0; n < NK; ++n) bf[n] = S[(JS * IR + (s * 4 + lc) * KB + n * 8 + lr) * PITCH];
            // the A fragments run FT_PF tiles ahead of the DMMAs that use them (explicit rotation: the compiler does not
            // move loads across the asm statements)
            const double* Ap = S + ((s * 4 + lc) * IR + lr) * PITCH;
            double afq[FT_PF];
#pragma unroll
            for (int m = 0; m < FT_PF; ++m) afq[m] = Ap[m * 8 * PITCH];
#pragma unroll
            for (int m = 0; m < FT_MT; ++m) {
                const double af = afq[m % FT_PF];
                if (m + FT_PF < FT_MT) afq[m % FT_PF] = Ap[(m + FT_PF) * 8 * PITCH];
#pragma unroll
                for (int n = 0; n < NK; ++n) dmma884k(acc[m][n][0], acc[m][n][1], af, bf[n]);
            }
        }
        if (!DIAG) {
            // direction 2: out[j][k] += sum_i tau[i][j] a[i][k], the 8 columns of this stage
            double acc2[NK][2];
#pragma unroll
            for (int n = 0; n < NK; ++n) { acc2[n][0] = 0.0; acc2[n][1] = 0.0; }
            const double* Atp = S + (lr * IR + lc) * PITCH;
            double atq[FT_PF];
#pragma unroll
            for (int q = 0; q < FT_PF; ++q) atq[q] = Atp[q * 4 * PITCH];
#pragma unroll
            for (int q = 0; q < IR / 4; ++q) {
                const double af = atq[q % FT_PF];
                if (q + FT_PF < IR / 4) atq[q % FT_PF] = Atp[(q + FT_PF) * 4 * PITCH];
#pragma unroll
                for (int n = 0; n < NK; ++n) dmma884k(acc2[n][0], acc2[n][1], af, breg[q][n]);
            }
#pragma unroll
            for (int n = 0; n < NK; ++n) {
                fl[(lr * KB + n * 8 + 2 * lc) * PITCH + w] = acc2[n][0];
                fl[(lr * KB + n * 8 + 2 * lc + 1) * PITCH + w] = acc2[n][1];
            }
            cp_async_wait<1>();          // this thread's out[J] pieces (the group before the next stage's copies)
            __syncthreads();
#pragma unroll
            for (int e = 0; e < NFL; ++e) {
                const int row = rsub + e * RSTEP, jj = row / KB, kk = row - jj * KB, col = js * JS + jj;
                if (row < JS * KB && col < tj && kk < kn) {
                    const double2 d = *(const double2*)(fl + row * PITCH + piece2);
                    const double2 o = *(const double2*)(ojs + row * PITCH + piece2);
                    *(double2*)(out_c + ((long)(j0 + col) * kc + kk) * CHUNK + piece2) = make_double2(fma(-alpha, d.x, o.x), fma(-alpha, d.y, o.y));
                }
            }
        }
    }
    // ---- epilogue: out[I] -= alpha * acc through shared memory (full rows)
    __syncthreads();
#pragma unroll
    for (int m = 0; m < FT_MT; ++m)
#pragma unroll
        for (int n = 0; n < NK; ++n) {
            sm[((m * 8 + lr) * KB + n * 8 + 2 * lc) * PITCH + w] = acc[m][n][0];
            sm[((m * 8 + lr) * KB + n * 8 + 2 * lc + 1) * PITCH + w] = acc[m][n][1];
        }
    __syncthreads();
    constexpr int EB = 14;               // rows in flight per thread: the loads of a batch are issued before its stores
    for (int row0 = rsub; row0 < ti * KB; row0 += EB * RSTEP) {
        double2 o[EB]; double* p[EB];
#pragma unroll
        for (int e = 0; e < EB; ++e) {
            const int row = row0 + e * RSTEP, i = row / KB, kk = row - i * KB;
            p[e] = (row < ti * KB && kk < kn) ? out_c + ((long)(i0 + i) * kc + kk) * CHUNK + piece2 : nullptr;
            o[e] = p[e] ? *(const double2*)p[e] : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int e = 0; e < EB; ++e) {
            if (p[e]) {
                const double2 d = *(const double2*)(sm + (row0 + e * RSTEP) * PITCH + piece2);
                *(double2*)p[e] = make_double2(fma(-alpha, d.x, o[e].x), fma(-alpha, d.y, o[e].y));
            }
        }
    }
}
template <int NK, bool DIAG, class SH>
static cudaError_t contract_full_launch(long nchunks, double* out, const double* a, const double* tau, int i0, int ti, int j0, int tj,
                                        int kc, int kn, long ftot, long stot, double alpha, cudaStream_t st) {
    constexpr size_t smem = FullCfg<NK, SH>::SMEM;
    static bool attr_done[kMaxDevices] = {false};
    const int dev = current_device();
    if (!attr_done[dev]) {
        cudaError_t e = cudaFuncSetAttribute(contract_full_kernel<NK, DIAG, SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_done[dev] = true;
    }
    contract_full_kernel<NK, DIAG, SH><<<(unsigned)(nchunks * (CHUNK / FT_P)), 32 * FT_P, smem, st>>>(out, a, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha);
    return cudaGetLastError();
}
int contract_full_max_tile() { return FullShapeL::TMAX; }
int contract_full_small_tile() { return FullShapeS::TMAX; }
template <class SH>
static cudaError_t contract_full_shape(bool diag, long nchunks, double* o, const double* ap, const double* tau, int i0, int ti, int j0, int tj,
                                       int kc, int kn, long ftot, long stot, double alpha, cudaStream_t st) {
    if (kn > 8) return diag ? contract_full_launch<2, true, SH>(nchunks, o, ap, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha, st)
                            : contract_full_launch<2, false, SH>(nchunks, o, ap, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha, st);
    return diag ? contract_full_launch<1, true, SH>(nchunks, o, ap, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha, st)
                : contract_full_launch<1, false, SH>(nchunks, o, ap, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha, st);
}
cudaError_t launch_contract_full(bool diag, double* out, const double* a, const double* tau, int i0, int ti, int j0, int tj, int kc,
                                 long ftot, long stot, long nr, double alpha, cudaStream_t st) {
    if (ti > FullShapeL::TMAX || tj < 1 || ti < 1 || (diag && ti != tj)) return cudaErrorInvalidValue;
    const long nchunks = (nr + CHUNK - 1) / CHUNK;
    for (int kb = 0; kb < kc; kb += 16) {
        const int kn = kc - kb < 16 ? kc - kb : 16;
        double* o = out + (long)kb * CHUNK; const double* ap = a + (long)kb * CHUNK;
        cudaError_t e = ti <= FullShapeS::TMAX ? contract_full_shape<FullShapeS>(diag, nchunks, o, ap, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha, st)
                                               : contract_full_shape<FullShapeL>(diag, nchunks, o, ap, tau, i0, ti, j0, tj, kc, kn, ftot, stot, alpha, st);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------------------
// V[kk][r] = f[r] * d[kk][r]: the spin-flip K1e potential f^SF * drho^SF (Eq. 24)
__global__ void scale_potential_kernel(const double* __restrict__ f, const double* __restrict__ d, long nr, double* __restrict__ V) {
    const long r = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (r >= nr) return;
    const long o = (long)blockIdx.y * nr + r;
    V[o] = f[r] * d[o];
}
cudaError_t launch_scale_potential(const double* f, const double* d, int kc, long nr, double* V, cudaStream_t st) {
    dim3 grid((unsigned)((nr + 255) / 256), (unsigned)kc);
    scale_potential_kernel<<<grid, 256, 0, st>>>(f, d, nr, V);
    return cudaGetLastError();
}

// D term alone (Eq. 3 with the kinetic model H): AX[f][g] = (kin[g] - eig[v]) X[f][g] for the functions of one spin block
__global__ void d_term_kernel(const cplx* __restrict__ X, cplx* __restrict__ AX, FunLayout lay, int nfun, const double* __restrict__ kin,
                              const double* __restrict__ eig) {
    const int f = blockIdx.y;
    const int v = f / lay.kc;
    const long o = (long)(lay.k0 + f % lay.kc) * lay.vec_len + lay.block_off + (long)v * lay.npwh;
    const double e = eig[v];
    for (long g = blockIdx.x * (long)blockDim.x + threadIdx.x; g < lay.npwh; g += (long)gridDim.x * blockDim.x) {
        const cplx x = X[o + g];
        const double d = kin[g] - e;
        AX[o + g] = make_double2(d * x.x, d * x.y);
    }
}
cudaError_t launch_d_term(const cplx* X, cplx* AX, FunLayout lay, int nfun, const double* kin, const double* eig, cudaStream_t st) {
    dim3 grid((unsigned)std::min<long>(64, (lay.npwh + 255) / 256), (unsigned)nfun);
    d_term_kernel<<<grid, 256, 0, st>>>(X, AX, lay, nfun, kin, eig);
    return cudaGetLastError();
}

// out[f0 + (t - t_first)*fstep][r] += scale * sum_{j < nj} M[j][r] * tau[j*nt + t][r],  t_first <= t < t_first + t_count
// (the sum over bands of Eq. 7 / Eq. 28: PAPER.md:95-96, :201-204).  M plain [j][nr]; tau chunked [nr/32][nj*nt][32];
// out chunked [nr/32][ftot][32].
template <int KT>
__global__ void pattern_reduce_kernel(const double* __restrict__ M, const double* __restrict__ tau, int nj, int nt, int t0, int tend, long nr,
                                      double* __restrict__ out, long ftot, long f0, long fstep, double scale) {
    const long r = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (r >= nr) return;
    double acc[KT];
#pragma unroll
    for (int q = 0; q < KT; ++q) acc[q] = 0.0;
    const double* tc = tau + (r >> 5) * ((long)nj * nt * CHUNK) + (r & (CHUNK - 1));
    for (int j = 0; j < nj; ++j) {
        const double m = M[(long)j * nr + r];
        const double* tj = tc + ((long)j * nt + t0) * CHUNK;
#pragma unroll
        for (int q = 0; q < KT; ++q) if (t0 + q < tend) acc[q] = fma(m, tj[q * CHUNK], acc[q]);
    }
    double* oc = out + (r >> 5) * (ftot * CHUNK) + (r & (CHUNK - 1));
#pragma unroll
    for (int q = 0; q < KT; ++q) if (t0 + q < tend) { double* o = oc + (f0 + (long)q * fstep) * CHUNK; *o = fma(scale, acc[q], *o); }
}
cudaError_t launch_pattern_reduce(const double* M, const double* tau, int nj, int nt, int t_first, int t_count, long nr, double* out, long ftot,
                                  long f0, long fstep, double scale, cudaStream_t st) {
    const unsigned nb = (unsigned)((nr + 127) / 128);
    for (int t0 = t_first; t0 < t_first + t_count; t0 += 4)
        pattern_reduce_kernel<4><<<nb, 128, 0, st>>>(M, tau, nj, nt, t0, t_first + t_count, nr, out, ftot, f0 + (long)(t0 - t_first) * fstep, fstep, scale);
    return cudaGetLastError();
}

// sq[v][r] = phi[v][r]^2 (the densities of Eq. 32)
__global__ void square_kernel(const double* __restrict__ phi, long n, double* __restrict__ sq) {
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) { const double p = phi[i]; sq[i] = p * p; }
}
cudaError_t launch_square(const double* phi, long n, double* sq, cudaStream_t st) {
    square_kernel<<<(unsigned)std::min<long>(65535, (n + 255) / 256), 256, 0, st>>>(phi, n, sq);
    return cudaGetLastError();
}

__global__ void symmetrize_kernel(double* __restrict__ H, int m, double scale) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m * m) return;
    const int r = i / m, c = i % m;
    if (r < c) { const double v = 0.5 * scale * (H[r * m + c] + H[c * m + r]); H[r * m + c] = v; H[c * m + r] = v; }
    else if (r == c) H[i] *= scale;
}
cudaError_t launch_symmetrize(double* H, int m, double scale, cudaStream_t st) {
    symmetrize_kernel<<<(m * m + 255) / 256, 256, 0, st>>>(H, m, scale);
    return cudaGetLastError();
}

// Cholesky A = L L^T of a small symmetric positive definite matrix and the inverse of L, one CTA, in global memory
// (ACE: M = -L L^T, xi = W L^-T, Eq. 30).  A [n][n] row-major is overwritten by L (lower triangle);
// Linv [n][n] receives L^-1 (lower triangular, zeros above).  status[0] = 0 or the 1-based index of a non-positive pivot.
__global__ void __launch_bounds__(1024) chol_inv_kernel(double* __restrict__ A, double* __restrict__ Linv, int n, int* __restrict__ status) {
    const int tid = threadIdx.x, nt = blockDim.x;
    __shared__ double piv;
    __shared__ int bad;
    if (tid == 0) bad = 0;
    __syncthreads();
    for (int k = 0; k < n; ++k) {
        if (tid == 0) { const double d = A[(long)k * n + k]; if (!(d > 0.0)) { bad = k + 1; piv = 1.0; } else piv = sqrt(d); }
        __syncthreads();
        if (bad) break;
        const double p = piv;
        for (int i = k + tid; i < n; i += nt) A[(long)i * n + k] = (i == k) ? p : A[(long)i * n + k] / p;
        __syncthreads();
        // trailing update of the lower triangle: A[i][j] -= L[i][k] L[j][k], k < j <= i
        const int m = n - k - 1;
        for (long e = tid; e < (long)m * m; e += nt) {
            const int i = k + 1 + (int)(e / m), j = k + 1 + (int)(e % m);
            if (j <= i) A[(long)i * n + j] -= A[(long)i * n + k] * A[(long)j * n + k];
        }
        __syncthreads();
    }
    if (tid == 0) status[0] = bad;
    if (bad) return;
    // columns of L^-1 by forward substitution, one column per thread: L x = e_c
    for (int c = tid; c < n; c += nt) {
        for (int i = 0; i < n; ++i) {
            if (i < c) { Linv[(long)i * n + c] = 0.0; continue; }
            double sacc = (i == c) ? 1.0 : 0.0;
            for (int j = c; j < i; ++j) sacc -= A[(long)i * n + j] * Linv[(long)j * n + c];
            Linv[(long)i * n + c] = sacc / A[(long)i * n + i];
        }
    }
}
cudaError_t launch_chol_inv(double* A, double* Linv, int n, int* status, cudaStream_t st) {
    chol_inv_kernel<<<1, 1024, 0, st>>>(A, Linv, n, status);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------
__global__ void rho0_kernel(const double* __restrict__ phi, int nocc, long nr, double* __restrict__ rho) {
    const long r = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (r >= nr) return;
    double s = 0.0;
    for (int v = 0; v < nocc; ++v) { const double p = phi[(long)v * nr + r]; s = fma(p, p, s); }
    rho[r] = s;
}
cudaError_t launch_rho0(const double* phi, int nocc, long nr, double* rho, cudaStream_t st) {
    rho0_kernel<<<(unsigned)((nr + 255) / 256), 256, 0, st>>>(phi, nocc, nr, rho);
    return cudaGetLastError();
}

// LDA: Slater exchange + Perdew-Zunger 1981 correlation, second derivatives written out by hand (reading A5).
// With E_c = rho eps(rs, zeta), eps = eU + f(zeta)(eP - eU), s_up = +1, s_dn = -1:
//   rho f_c,ss' = -(rs/3)(2/3 eps_rs - rs/3 eps_rsrs) - (rs/3) eps_rszeta (s + s' - 2 zeta) + (s - zeta)(s' - zeta) eps_zetazeta
struct PZ { double gamma, beta1, beta2, A, B, C, D; };
__device__ __forceinline__ void pz_eps(const PZ& p, double rs, double& e, double& e1, double& e2) {
    if (rs >= 1.0) {
        const double sq = sqrt(rs);
        const double Dn = 1.0 + p.beta1 * sq + p.beta2 * rs;
        const double D1 = 0.5 * p.beta1 / sq + p.beta2;
        const double D2 = -0.25 * p.beta1 / (rs * sq);
        e = p.gamma / Dn;
        e1 = -p.gamma * D1 / (Dn * Dn);
        e2 = -p.gamma * D2 / (Dn * Dn) + 2.0 * p.gamma * D1 * D1 / (Dn * Dn * Dn);
    } else {
        const double l = log(rs);
        e = p.A * l + p.B + p.C * rs * l + p.D * rs;
        e1 = p.A / rs + p.C * (l + 1.0) + p.D;
        e2 = -p.A / (rs * rs) + p.C / rs;
    }
}
__global__ void lda_fxc_kernel(const double* __restrict__ rho_up, const double* __restrict__ rho_dn, long nr, double rho_floor,
                               double* __restrict__ fuu, double* __restrict__ fud, double* __restrict__ fdd) {
    const long r = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (r >= nr) return;
    const double ru = rho_up[r], rd = rho_dn[r];
    if (!(ru >= rho_floor) || !(rd >= rho_floor)) { fuu[r] = 0.0; fud[r] = 0.0; fdd[r] = 0.0; return; }
    const double cx = -(1.0 / 3.0) * cbrt(6.0 / M_PI);
    const double fxu = cx / (cbrt(ru) * cbrt(ru)), fxd = cx / (cbrt(rd) * cbrt(rd));
    const double rho = ru + rd, zeta = (ru - rd) / rho;
    const double rs = cbrt(3.0 / (4.0 * M_PI * rho));
    const PZ U = {-0.1423, 1.0529, 0.3334, 0.0311, -0.048, 0.0020, -0.0116};
    const PZ P = {-0.0843, 1.3981, 0.2611, 0.01555, -0.0269, 0.0007, -0.0048};
    double eu, eu1, eu2, ep, ep1, ep2;
    pz_eps(U, rs, eu, eu1, eu2);
    pz_eps(P, rs, ep, ep1, ep2);
    const double c0 = 2.0 * cbrt(2.0) - 2.0;                 // 2^(4/3) - 2
    const double op = cbrt(1.0 + zeta), om = cbrt(1.0 - zeta);
    const double fz = (op * op * op * op + om * om * om * om - 2.0) / c0;
    const double fz1 = (4.0 / 3.0) * (op - om) / c0;
    const double fz2 = (4.0 / 9.0) * (1.0 / (op * op) + 1.0 / (om * om)) / c0;
    const double d = ep - eu, d1 = ep1 - eu1, d2 = ep2 - eu2;
    const double e_rs = eu1 + fz * d1, e_rsrs = eu2 + fz * d2;
    const double e_rsz = fz1 * d1, e_zz = fz2 * d;
    const double base = -(rs / 3.0) * ((2.0 / 3.0) * e_rs - (rs / 3.0) * e_rsrs);
    const double cross = -(rs / 3.0) * e_rsz;
    const double su = 1.0 - zeta, sd = -1.0 - zeta;
    fuu[r] = fxu + (base + cross * (2.0 - 2.0 * zeta) + su * su * e_zz) / rho;
    fud[r] = (base + cross * (-2.0 * zeta) + su * sd * e_zz) / rho;
    fdd[r] = fxd + (base + cross * (-2.0 - 2.0 * zeta) + sd * sd * e_zz) / rho;
}
cudaError_t launch_lda_fxc(const double* rho_up, const double* rho_dn, long nr, double rho_floor, double* fuu, double* fud,
                           double* fdd, cudaStream_t st) {
    lda_fxc_kernel<<<(unsigned)((nr + 255) / 256), 256, 0, st>>>(rho_up, rho_dn, nr, rho_floor, fuu, fud, fdd);
    return cudaGetLastError();
}

// Spin-flip xc kernel of Eq. 26: f^SF = (V_xc,up - V_xc,dn) / (rho_up - rho_dn), zero where
// |rho_up - rho_dn| < cut.  V_xc by hand: v_x,s = -(6 rho_s/pi)^(1/3);
// v_c,s = eps - (rs/3) eps_rs + (s - zeta) eps_zeta, so v_c,up - v_c,dn = 2 eps_zeta = 2 f'(zeta) (eps_P - eps_U).
// The potentials are evaluated at densities clamped from below at rho_floor (reading A5).
__global__ void sf_kernel_table(const double* __restrict__ rho_up, const double* __restrict__ rho_dn, long nr, double rho_floor,
                                double cut, double* __restrict__ fsf) {
    const long r = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (r >= nr) return;
    const double d = rho_up[r] - rho_dn[r];
    if (!(fabs(d) >= cut)) { fsf[r] = 0.0; return; }
    const double ru = fmax(rho_up[r], rho_floor), rd = fmax(rho_dn[r], rho_floor);
    const double rho = ru + rd, zeta = (ru - rd) / rho;
    const double rs = cbrt(3.0 / (4.0 * M_PI * rho));
    const PZ U = {-0.1423, 1.0529, 0.3334, 0.0311, -0.048, 0.0020, -0.0116};
    const PZ P = {-0.0843, 1.3981, 0.2611, 0.01555, -0.0269, 0.0007, -0.0048};
    double eu, eu1, eu2, ep, ep1, ep2;
    pz_eps(U, rs, eu, eu1, eu2);
    pz_eps(P, rs, ep, ep1, ep2);
    const double c0 = 2.0 * cbrt(2.0) - 2.0;
    const double fz1 = (4.0 / 3.0) * (cbrt(1.0 + zeta) - cbrt(1.0 - zeta)) / c0;
    const double dvx = -cbrt(6.0 / M_PI) * (cbrt(ru) - cbrt(rd));
    fsf[r] = (dvx + 2.0 * fz1 * (ep - eu)) / d;
}
cudaError_t launch_sf_kernel_table(const double* rho_up, const double* rho_dn, long nr, double rho_floor, double cut, double* fsf,
                                   cudaStream_t st) {
    sf_kernel_table<<<(unsigned)((nr + 255) / 256), 256, 0, st>>>(rho_up, rho_dn, nr, rho_floor, cut, fsf);
    return cudaGetLastError();
}

}  // namespace tddft
