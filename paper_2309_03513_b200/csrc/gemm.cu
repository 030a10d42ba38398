// Dense FP64 contractions on the tensor cores (DMMA, mma.sync.m8n8k4.f64): the conduction-band projector
// P_c = 1 - sum_v |phi_v><phi_v| and the Davidson subspace matrices.
// tcgen05 has no FP64 path, so the FP64 tensor pipe is reached through mma.sync; measured DMMA peak on B200 equals
// the DFMA peak (36.9 TFLOP/s), the gain is issue slots and register traffic, not raw rate.
#include "kernels.h"
#include "gemm_pipe.cuh"

namespace tddft {

constexpr int BM = 64, BN = 64, BK = 16, LDS = 68;   // LDS % 16 == 4: conflict-free fragment reads

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// one BK slab: warp (wm, wn) owns a 32x32 block = 4x4 fragments
__device__ __forceinline__ void mma_slab(const double (*As)[LDS], const double (*Bs)[LDS], int wm, int wn, int lane,
                                         double (&acc)[4][4][2]) {
    const int lr = lane >> 2, lc = lane & 3;
#pragma unroll
    for (int k0 = 0; k0 < BK; k0 += 4) {
        double af[4], bf[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) af[i] = As[k0 + lc][wm * 32 + i * 8 + lr];
#pragma unroll
        for (int j = 0; j < 4; ++j) bf[j] = Bs[k0 + lc][wn * 32 + j * 8 + lr];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
    }
}

__global__ void __launch_bounds__(128) gemm_nt_kernel(const double* __restrict__ A, long lda, const double* __restrict__ B, long ldb,
                                                      int bgrp, long bstride_grp, double* __restrict__ C, long ldc, int M, int N,
                                                      long K, long kper, long wperiod, double cscale, int splits,
                                                      double* __restrict__ partial) {
    __shared__ double As[BK][LDS], Bs[BK][LDS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, wm = warp >> 1, wn = warp & 1;
    const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
    const long kbeg = (long)blockIdx.z * kper, kend = min(K, kbeg + kper);
    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    const int row = tid >> 1, kh = (tid & 1) * 8;
    const double* arow = (m0 + row < M) ? A + (long)(m0 + row) * lda : nullptr;
    const int nb = n0 + row;
    const double* brow = (nb < N) ? B + (long)(nb / bgrp) * bstride_grp + (long)(nb % bgrp) * ldb : nullptr;
    for (long k0 = kbeg; k0 < kend; k0 += BK) {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const long k = k0 + kh + q;
            double a = (arow && k < kend) ? arow[k] : 0.0;
            if (wperiod > 0 && (k % wperiod) == 0) a *= 0.5;
            As[kh + q][row] = a;
            Bs[kh + q][row] = (brow && k < kend) ? brow[k] : 0.0;
        }
        __syncthreads();
        mma_slab(As, Bs, wm, wn, lane, acc);
        __syncthreads();
    }
    const int lr = lane >> 2, lc = lane & 3;
    double* dst = (splits > 1) ? partial + (long)blockIdx.z * M * N : C;
    const long ld = (splits > 1) ? N : ldc;
    const double sc = (splits > 1) ? 1.0 : cscale;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int m = m0 + wm * 32 + i * 8 + lr, n = n0 + wn * 32 + j * 8 + 2 * lc;
            if (m < M) {
                if (n < N) dst[(long)m * ld + n] = sc * acc[i][j][0];
                if (n + 1 < N) dst[(long)m * ld + n + 1] = sc * acc[i][j][1];
            }
        }
}
__global__ void splitk_reduce_kernel(const double* __restrict__ partial, int splits, long mn, int N, double* __restrict__ C, long ldc,
                                     double cscale) {
    const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i >= mn) return;
    double s = 0.0;
    for (int z = 0; z < splits; ++z) s += partial[(long)z * mn + i];
    C[(i / N) * ldc + (i % N)] = cscale * s;
}
template <class CFG>
static cudaError_t nt_pipe_launch(const double* A, long lda, const double* B, long ldb, int bgrp, long bstride_grp, double* C, long ldc,
                                  int M, int N, long K, long kper, long wperiod, double cscale, int splits, double* partial, cudaStream_t st) {
    static bool attr_done[kMaxDevices] = {false};
    const int dev = current_device();
    if (!attr_done[dev]) {
        cudaError_t e = cudaFuncSetAttribute(gemm_nt_pipe_kernel<CFG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CFG::SMEM_NT);
        if (e != cudaSuccess) return e;
        attr_done[dev] = true;
    }
    dim3 grid((unsigned)((N + CFG::BN - 1) / CFG::BN), (unsigned)((M + CFG::BM - 1) / CFG::BM), (unsigned)splits);
    gemm_nt_pipe_kernel<CFG><<<grid, CFG::NTHR, CFG::SMEM_NT, st>>>(A, lda, B, ldb, bgrp, bstride_grp, C, ldc, M, N, K, kper, wperiod, cscale, splits, partial);
    return cudaGetLastError();
}
typedef GemmCfg<144, 128, 72, 32, 4> NtBig;     // orbitals x functions: 432 = 3 x 144, 1150 ~ 8 x 144
typedef GemmCfg<64, 64, 32, 32, 4> NtSmall;     // Davidson Gram matrices (m <= a few hundred, K = 10^7)
typedef GemmCfg<128, 72, 32, 72, 4, 2> TnBig;    // two 4-warp CTAs per SM: one epilogue (C read-modify-write) runs behind the other DMMAs

int gemm_nt_tile_count(int M, int N) {
    if (M >= 96 && N >= 96) return ((M + NtBig::BM - 1) / NtBig::BM) * ((N + NtBig::BN - 1) / NtBig::BN);
    return ((M + 63) / 64) * ((N + 63) / 64);
}
cudaError_t launch_gemm_nt(const double* A, long lda, const double* B, long ldb, int bgrp, long bstride_grp, double* C, long ldc,
                           int M, int N, long K, long wperiod, double cscale, int splits, double* partial, cudaStream_t st) {
    if (splits < 1 || !partial) splits = 1;
    long kper = ((K + splits - 1) / splits + BK - 1) / BK * BK;
    splits = (int)((K + kper - 1) / kper);
    const bool aligned = (lda % 2 == 0) && (ldb % 2 == 0) && (bstride_grp % 2 == 0) && (((size_t)A | (size_t)B) % 16 == 0);
    cudaError_t e;
    if (!aligned) {
        dim3 grid((unsigned)((N + BN - 1) / BN), (unsigned)((M + BM - 1) / BM), (unsigned)splits);
        gemm_nt_kernel<<<grid, 128, 0, st>>>(A, lda, B, ldb, bgrp, bstride_grp, C, ldc, M, N, K, kper, wperiod, cscale, splits, partial);
        e = cudaGetLastError();
    } else if (M >= 96 && N >= 96) {
        e = nt_pipe_launch<NtBig>(A, lda, B, ldb, bgrp, bstride_grp, C, ldc, M, N, K, kper, wperiod, cscale, splits, partial, st);
    } else {
        e = nt_pipe_launch<NtSmall>(A, lda, B, ldb, bgrp, bstride_grp, C, ldc, M, N, K, kper, wperiod, cscale, splits, partial, st);
    }
    if (e != cudaSuccess) return e;
    if (splits > 1) {
        const long mn = (long)M * N;
        splitk_reduce_kernel<<<(unsigned)((mn + 255) / 256), 256, 0, st>>>(partial, splits, mn, N, C, ldc, cscale);
    }
    return cudaGetLastError();
}

cudaError_t launch_gram_shift(const double* Phi, long lda, int M, long K, const double* kin, const double* lam, int nb, double dfloor,
                              double* S, cudaStream_t st) {
    if (lda % 2 != 0 || ((size_t)Phi) % 16 != 0) return cudaErrorInvalidValue;
    dim3 grid;
    if (M >= 96) {
        static bool attr_done[kMaxDevices] = {false};
        const int dev = current_device();
        if (!attr_done[dev]) {
            cudaError_t e = cudaFuncSetAttribute(gram_shift_kernel<NtBig>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)NtBig::SMEM_NT);
            if (e != cudaSuccess) return e;
            attr_done[dev] = true;
        }
        grid = dim3((unsigned)((M + NtBig::BN - 1) / NtBig::BN), (unsigned)((M + NtBig::BM - 1) / NtBig::BM), (unsigned)nb);
        gram_shift_kernel<NtBig><<<grid, NtBig::NTHR, NtBig::SMEM_NT, st>>>(Phi, lda, M, K, kin, lam, dfloor, S);
    } else {
        static bool attr_done[kMaxDevices] = {false};
        const int dev = current_device();
        if (!attr_done[dev]) {
            cudaError_t e = cudaFuncSetAttribute(gram_shift_kernel<NtSmall>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)NtSmall::SMEM_NT);
            if (e != cudaSuccess) return e;
            attr_done[dev] = true;
        }
        grid = dim3((unsigned)((M + NtSmall::BN - 1) / NtSmall::BN), (unsigned)((M + NtSmall::BM - 1) / NtSmall::BM), (unsigned)nb);
        gram_shift_kernel<NtSmall><<<grid, NtSmall::NTHR, NtSmall::SMEM_NT, st>>>(Phi, lda, M, K, kin, lam, dfloor, S);
    }
    return cudaGetLastError();
}

__global__ void __launch_bounds__(128) gemm_tn_acc_kernel(const double* __restrict__ At, long ldat, const double* __restrict__ B, long ldb,
                                                          double* __restrict__ C, long ldc, int cgrp, long cstride_grp, int M, long N,
                                                          int K, double cscale) {
    __shared__ double As[BK][LDS], Bs[BK][LDS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, wm = warp >> 1, wn = warp & 1;
    const int m0 = blockIdx.y * BM;
    const long n0 = (long)blockIdx.x * BN;
    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    const int kr = tid >> 3, c8 = (tid & 7) * 8;    // 16 rows x 8 threads, 8 consecutive doubles each
    for (int k0 = 0; k0 < K; k0 += BK) {
        const int k = k0 + kr;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int m = m0 + c8 + q;
            As[kr][c8 + q] = (k < K && m < M) ? At[(long)k * ldat + m] : 0.0;
            const long n = n0 + c8 + q;
            Bs[kr][c8 + q] = (k < K && n < N) ? B[(long)k * ldb + n] : 0.0;
        }
        __syncthreads();
        mma_slab(As, Bs, wm, wn, lane, acc);
        __syncthreads();
    }
    const int lr = lane >> 2, lc = lane & 3;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int m = m0 + wm * 32 + i * 8 + lr;
        if (m >= M) continue;
        double* crow = C + (long)(m / cgrp) * cstride_grp + (long)(m % cgrp) * ldc;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const long n = n0 + wn * 32 + j * 8 + 2 * lc;
            if (n < N) crow[n] = fma(cscale, acc[i][j][0], crow[n]);
            if (n + 1 < N) crow[n + 1] = fma(cscale, acc[i][j][1], crow[n + 1]);
        }
    }
}
cudaError_t launch_gemm_tn_acc(const double* At, long ldat, const double* B, long ldb, double* C, long ldc, int cgrp,
                               long cstride_grp, int M, long N, int K, double cscale, cudaStream_t st) {
    const bool aligned = (ldat % 2 == 0) && (ldb % 2 == 0) && (((size_t)At | (size_t)B) % 16 == 0);
    if (aligned && M >= 96 && N >= 96) {
        static bool attr_done[kMaxDevices] = {false};
        const int dev = current_device();
        if (!attr_done[dev]) {
            cudaError_t e = cudaFuncSetAttribute(gemm_tn_pipe_kernel<TnBig>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TnBig::SMEM_TN);
            if (e != cudaSuccess) return e;
            attr_done[dev] = true;
        }
        dim3 grid((unsigned)((N + TnBig::BN - 1) / TnBig::BN), (unsigned)((M + TnBig::BM - 1) / TnBig::BM));
        gemm_tn_pipe_kernel<TnBig><<<grid, TnBig::NTHR, TnBig::SMEM_TN, st>>>(At, ldat, B, ldb, C, ldc, cgrp, cstride_grp, M, N, K, cscale);
        return cudaGetLastError();
    }
    dim3 grid((unsigned)((N + BN - 1) / BN), (unsigned)((M + BM - 1) / BM));
    gemm_tn_acc_kernel<<<grid, 128, 0, st>>>(At, ldat, B, ldb, C, ldc, cgrp, cstride_grp, M, N, K, cscale);
    return cudaGetLastError();
}

}  // namespace tddft
