// Pipelined FP64 tensor-core GEMM tiles (mma.sync.m8n8k4.f64, "DMMA"; tcgen05 has no FP64 path) for the dense
// contractions of the hot path: the conduction-band projector P_c = 1 - sum_v |phi_v><phi_v| (PAPER.md:105,
// SURVEY S8) and the Davidson overlap / subspace matrices.
// Operands stream global -> shared through a multi-stage cp.async ring (16-byte copies, zero-filled tails), so
// the DMMA pipe never waits for a load phase; fragment reads are bank-conflict free by row padding (pitch = 4 mod 16).
#pragma once
#include <cuda_runtime.h>

namespace tddft {

constexpr int GK = 16;          // k extent of one stage

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
// 16-byte async copy, `bytes` (0, 8 or 16) valid, the rest zero-filled
__device__ __forceinline__ void cp16z(void* smem, const void* gmem, int bytes) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(sa), "l"(gmem), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int BM_, int BN_, int WM_, int WN_, int STAGES_, int MINB_ = 1> struct GemmCfg {
    static constexpr int BM = BM_, BN = BN_, WM = WM_, WN = WN_, STAGES = STAGES_, MINB = MINB_;   // MINB: CTAs per SM
    static constexpr int WARPS_M = BM / WM, WARPS_N = BN / WN, NTHR = 32 * WARPS_M * WARPS_N;
    static constexpr int FM = WM / 8, FN = WN / 8;
    // NT: rows K-contiguous, pitch GK + 4;  TN: rows M/N-contiguous, pitch = 4 mod 16
    static constexpr int LDK = GK + 4;
    static constexpr int LDM = BM + ((4 - BM % 16) + 16) % 16, LDN = BN + ((4 - BN % 16) + 16) % 16;
    static constexpr size_t SMEM_NT = sizeof(double) * STAGES * (BM + BN) * LDK;
    static constexpr size_t SMEM_TN = sizeof(double) * STAGES * GK * (LDM + LDN);
};

// C[m][n] (ldc) = cscale * sum_k w_k A[m][k] B[n][k];  B row n at B + (n / bgrp)*bstride_grp + (n % bgrp)*ldb.
// w_k = 1/2 for k % wperiod == 0 (wperiod > 0), applied as a correction after the main loop.
// blockIdx.z = k split; with splits > 1 the raw partial sums go to partial[z][M][N].
template <class CFG>
__global__ void __launch_bounds__(CFG::NTHR, 1)
gemm_nt_pipe_kernel(const double* __restrict__ A, long lda, const double* __restrict__ B, long ldb, int bgrp, long bstride_grp,
                    double* __restrict__ C, long ldc, int M, int N, long K, long kper, long wperiod, double cscale, int splits,
                    double* __restrict__ partial) {
    constexpr int BM = CFG::BM, BN = CFG::BN, LDK = CFG::LDK, ST = CFG::STAGES, NTHR = CFG::NTHR, FM = CFG::FM, FN = CFG::FN;
    extern __shared__ __align__(16) double gsm[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm0 = (warp / CFG::WARPS_N) * CFG::WM, wn0 = (warp % CFG::WARPS_N) * CFG::WN;
    const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
    const long kbeg = (long)blockIdx.z * kper, kend = min(K, kbeg + kper);
    const int KT = (int)((kend - kbeg + GK - 1) / GK);
    constexpr int CHUNKS = (BM + BN) * (GK / 2);          // 16-byte chunks per stage
    constexpr int NQ = (CHUNKS + NTHR - 1) / NTHR;
    const double* src[NQ]; int soff[NQ]; int kc2[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int ch = tid + q * NTHR;
        const int row = ch / (GK / 2), kc = (ch % (GK / 2)) * 2;
        src[q] = nullptr; soff[q] = row * LDK + kc; kc2[q] = kc;
        if (ch < CHUNKS) {
            if (row < BM) { if (m0 + row < M) src[q] = A + (long)(m0 + row) * lda + kbeg + kc; }
            else { const int n = n0 + row - BM; if (n < N) src[q] = B + (long)(n / bgrp) * bstride_grp + (long)(n % bgrp) * ldb + kbeg + kc; }
        } else soff[q] = -1;
    }
    auto load_stage = [&](int buf, int kt) {
        double* base = gsm + (size_t)buf * (BM + BN) * LDK;
        const long krem = kend - kbeg - (long)kt * GK;     // valid k in this stage (may exceed GK)
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            if (soff[q] < 0) continue;
            long left = krem - kc2[q];
            int bytes = (src[q] && left > 0) ? (left >= 2 ? 16 : 8) : 0;
            cp16z(base + soff[q], bytes ? (const void*)(src[q] + (long)kt * GK) : (const void*)A, bytes);
        }
    };
    double acc[FM][FN][2];
#pragma unroll
    for (int i = 0; i < FM; ++i)
#pragma unroll
        for (int j = 0; j < FN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
#pragma unroll
    for (int s = 0; s < ST - 1; ++s) { if (s < KT) load_stage(s, s); cp_commit(); }
    const int lr = lane >> 2, lc = lane & 3;
    for (int kt = 0; kt < KT; ++kt) {
        cp_wait<ST - 2>();
        __syncthreads();
        if (kt + ST - 1 < KT) load_stage((kt + ST - 1) % ST, kt + ST - 1);
        cp_commit();
        const double* As = gsm + (size_t)(kt % ST) * (BM + BN) * LDK + (wm0 + lr) * LDK + lc;
        const double* Bs = gsm + (size_t)(kt % ST) * (BM + BN) * LDK + (BM + wn0 + lr) * LDK + lc;
#pragma unroll
        for (int k0 = 0; k0 < GK; k0 += 4) {
            double af[FM], bf[FN];
#pragma unroll
            for (int i = 0; i < FM; ++i) af[i] = As[i * 8 * LDK + k0];
#pragma unroll
            for (int j = 0; j < FN; ++j) bf[j] = Bs[j * 8 * LDK + k0];
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) dmma(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
    }
    cp_wait<0>();
    double* dst = (splits > 1) ? partial + (long)blockIdx.z * M * N : C;
    const long ld = (splits > 1) ? N : ldc;
    const double sc = (splits > 1) ? 1.0 : cscale;
    long kw = -1;
    if (wperiod > 0) { kw = (kbeg + wperiod - 1) / wperiod * wperiod; if (kw >= kend) kw = -1; }
#pragma unroll
    for (int i = 0; i < FM; ++i) {
        const int m = m0 + wm0 + i * 8 + lr;
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < FN; ++j)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int n = n0 + wn0 + j * 8 + 2 * lc + h;
                if (n >= N) continue;
                double v = acc[i][j][h];
                if (kw >= 0) {
                    const double* brow = B + (long)(n / bgrp) * bstride_grp + (long)(n % bgrp) * ldb;
                    for (long k = kw; k < kend; k += wperiod) v = fma(-0.5 * A[(long)m * lda + k], brow[k], v);
                }
                dst[(long)m * ld + n] = sc * v;
            }
    }
}

// C[m][n] += cscale * sum_k At[k][m] B[k][n];  C row m at C + (m / cgrp)*cstride_grp + (m % cgrp)*ldc.
// At rows (ldat) and B rows (ldb) must start 16-byte aligned (ldat, ldb even).
template <class CFG>
__global__ void __launch_bounds__(CFG::NTHR, CFG::MINB)
gemm_tn_pipe_kernel(const double* __restrict__ At, long ldat, const double* __restrict__ B, long ldb, double* __restrict__ C, long ldc,
                    int cgrp, long cstride_grp, int M, long N, int K, double cscale) {
    constexpr int BM = CFG::BM, BN = CFG::BN, LDM = CFG::LDM, LDN = CFG::LDN, ST = CFG::STAGES, NTHR = CFG::NTHR, FM = CFG::FM, FN = CFG::FN;
    extern __shared__ __align__(16) double gsm[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm0 = (warp / CFG::WARPS_N) * CFG::WM, wn0 = (warp % CFG::WARPS_N) * CFG::WN;
    const int m0 = blockIdx.y * BM;
    const long n0 = (long)blockIdx.x * BN;
    const int KT = (K + GK - 1) / GK;
    constexpr int CA = GK * (BM / 2), CB = GK * (BN / 2), CHUNKS = CA + CB;
    constexpr int NQ = (CHUNKS + NTHR - 1) / NTHR;
    const double* src[NQ]; int soff[NQ]; int krow[NQ]; int bytes0[NQ]; long kstride[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int ch = tid + q * NTHR;
        src[q] = nullptr; soff[q] = -1; krow[q] = 0; bytes0[q] = 0; kstride[q] = 0;
        if (ch < CA) {
            const int k = ch / (BM / 2), c2 = (ch % (BM / 2)) * 2;
            const long left = (long)M - (m0 + c2);
            krow[q] = k; soff[q] = k * LDM + c2; kstride[q] = ldat;
            bytes0[q] = left >= 2 ? 16 : (left == 1 ? 8 : 0);
            src[q] = At + (long)k * ldat + m0 + c2;
        } else if (ch < CHUNKS) {
            const int cb = ch - CA;
            const int k = cb / (BN / 2), c2 = (cb % (BN / 2)) * 2;
            const long left = N - (n0 + c2);
            krow[q] = k; soff[q] = GK * LDM + k * LDN + c2; kstride[q] = ldb;
            bytes0[q] = left >= 2 ? 16 : (left == 1 ? 8 : 0);
            src[q] = B + (long)k * ldb + n0 + c2;
        }
    }
    auto load_stage = [&](int buf, int kt) {
        double* base = gsm + (size_t)buf * GK * (LDM + LDN);
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            if (soff[q] < 0) continue;
            const int bytes = (kt * GK + krow[q] < K) ? bytes0[q] : 0;
            cp16z(base + soff[q], bytes ? (const void*)(src[q] + (long)kt * GK * kstride[q]) : (const void*)At, bytes);
        }
    };
    double acc[FM][FN][2];
#pragma unroll
    for (int i = 0; i < FM; ++i)
#pragma unroll
        for (int j = 0; j < FN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
#pragma unroll
    for (int s = 0; s < ST - 1; ++s) { if (s < KT) load_stage(s, s); cp_commit(); }
    const int lr = lane >> 2, lc = lane & 3;
    for (int kt = 0; kt < KT; ++kt) {
        cp_wait<ST - 2>();
        __syncthreads();
        if (kt + ST - 1 < KT) load_stage((kt + ST - 1) % ST, kt + ST - 1);
        cp_commit();
        const double* As = gsm + (size_t)(kt % ST) * GK * (LDM + LDN) + lc * LDM + wm0 + lr;
        const double* Bs = gsm + (size_t)(kt % ST) * GK * (LDM + LDN) + GK * LDM + lc * LDN + wn0 + lr;
#pragma unroll
        for (int k0 = 0; k0 < GK; k0 += 4) {
            double af[FM], bf[FN];
#pragma unroll
            for (int i = 0; i < FM; ++i) af[i] = As[k0 * LDM + i * 8];
#pragma unroll
            for (int j = 0; j < FN; ++j) bf[j] = Bs[k0 * LDN + j * 8];
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) dmma(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
    }
    cp_wait<0>();
#pragma unroll
    for (int i = 0; i < FM; ++i) {
        const int m = m0 + wm0 + i * 8 + lr;
        if (m >= M) continue;
        double* crow = C + (long)(m / cgrp) * cstride_grp + (long)(m % cgrp) * ldc;
#pragma unroll
        for (int j = 0; j < FN; ++j) {
            const long n = n0 + wn0 + j * 8 + 2 * lc;
            if (n + 1 < N) {
                double2* p = (double2*)(crow + n);
                if ((((size_t)p) & 15) == 0) { double2 v = *p; v.x = fma(cscale, acc[i][j][0], v.x); v.y = fma(cscale, acc[i][j][1], v.y); *p = v; }
                else { crow[n] = fma(cscale, acc[i][j][0], crow[n]); crow[n + 1] = fma(cscale, acc[i][j][1], crow[n + 1]); }
            } else if (n < N) crow[n] = fma(cscale, acc[i][j][0], crow[n]);
        }
    }
}

// Shifted, weighted Gram matrices of the projector-aware Davidson correction (reading A11b of DESIGN.md):
//   S_b[u][u'] = sum_k Phi[u][k] Phi[u'][k] w_b[k],   w_b[k] = gamma_k / d,  d = kin[k/2] - lam[b] with |d| floored at dfloor (sign kept),
// gamma_k = 2 (1 for Re c(G=0), 0 for Im c(G=0)): the Gamma inner product of <phi_u| (T - lambda)^-1 |phi_u'>.
// Phi [M][K] K-contiguous (K = 2 npwh reals); blockIdx.z = b; S [nb][M][M].  Same pipeline as gemm_nt_pipe_kernel, the weight is
// applied to the B fragments in registers.
template <class CFG>
__global__ void __launch_bounds__(CFG::NTHR, 1)
gram_shift_kernel(const double* __restrict__ A, long lda, int M, long K, const double* __restrict__ kin, const double* __restrict__ lam,
                  double dfloor, double* __restrict__ S) {
    constexpr int BM = CFG::BM, BN = CFG::BN, LDK = CFG::LDK, ST = CFG::STAGES, NTHR = CFG::NTHR, FM = CFG::FM, FN = CFG::FN;
    extern __shared__ __align__(16) double gsm[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm0 = (warp / CFG::WARPS_N) * CFG::WM, wn0 = (warp % CFG::WARPS_N) * CFG::WN;
    const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
    const double lambda = lam[blockIdx.z];
    const int KT = (int)((K + GK - 1) / GK);
    constexpr int CHUNKS = (BM + BN) * (GK / 2);
    constexpr int NQ = (CHUNKS + NTHR - 1) / NTHR;
    const double* src[NQ]; int soff[NQ]; int kc2[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int ch = tid + q * NTHR;
        const int row = ch / (GK / 2), kc = (ch % (GK / 2)) * 2;
        src[q] = nullptr; soff[q] = row * LDK + kc; kc2[q] = kc;
        if (ch < CHUNKS) {
            const int r = row < BM ? m0 + row : n0 + row - BM;
            if (r < M) src[q] = A + (long)r * lda + kc;
        } else soff[q] = -1;
    }
    auto load_stage = [&](int buf, int kt) {
        double* base = gsm + (size_t)buf * (BM + BN) * LDK;
        const long krem = K - (long)kt * GK;
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            if (soff[q] < 0) continue;
            long left = krem - kc2[q];
            int bytes = (src[q] && left > 0) ? (left >= 2 ? 16 : 8) : 0;
            cp16z(base + soff[q], bytes ? (const void*)(src[q] + (long)kt * GK) : (const void*)A, bytes);
        }
    };
    double acc[FM][FN][2];
#pragma unroll
    for (int i = 0; i < FM; ++i)
#pragma unroll
        for (int j = 0; j < FN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
#pragma unroll
    for (int s = 0; s < ST - 1; ++s) { if (s < KT) load_stage(s, s); cp_commit(); }
    const int lr = lane >> 2, lc = lane & 3;
    for (int kt = 0; kt < KT; ++kt) {
        // this lane's weights of the stage: k = kt*GK + k0 + lc
        double w[GK / 4];
#pragma unroll
        for (int q = 0; q < GK / 4; ++q) {
            const long k = (long)kt * GK + q * 4 + lc;
            double wv = 0.0;
            if (k < K) {
                double d = __ldg(kin + (k >> 1)) - lambda;
                if (fabs(d) < dfloor) d = d < 0 ? -dfloor : dfloor;
                wv = (k >= 2) ? 2.0 / d : (k == 0 ? 1.0 / d : 0.0);
            }
            w[q] = wv;
        }
        cp_wait<ST - 2>();
        __syncthreads();
        if (kt + ST - 1 < KT) load_stage((kt + ST - 1) % ST, kt + ST - 1);
        cp_commit();
        const double* As = gsm + (size_t)(kt % ST) * (BM + BN) * LDK + (wm0 + lr) * LDK + lc;
        const double* Bs = gsm + (size_t)(kt % ST) * (BM + BN) * LDK + (BM + wn0 + lr) * LDK + lc;
#pragma unroll
        for (int k0 = 0; k0 < GK; k0 += 4) {
            double af[FM], bf[FN];
#pragma unroll
            for (int i = 0; i < FM; ++i) af[i] = As[i * 8 * LDK + k0];
#pragma unroll
            for (int j = 0; j < FN; ++j) bf[j] = Bs[j * 8 * LDK + k0] * w[k0 / 4];
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) dmma(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
    }
    cp_wait<0>();
    double* dst = S + (size_t)blockIdx.z * M * M;
#pragma unroll
    for (int i = 0; i < FM; ++i) {
        const int m = m0 + wm0 + i * 8 + lr;
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < FN; ++j)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int n = n0 + wn0 + j * 8 + 2 * lc + h;
                if (n < M) dst[(long)m * M + n] = acc[i][j][h];
            }
    }
}

}  // namespace tddft
