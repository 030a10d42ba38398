// Block Davidson-Liu driver for the lowest roots of the TDA operator (PAPER.md:274 says only
// "The diagonalization is carried out iteratively using the Davidson method", ref. 85; the algorithm is
// reading A11 of DESIGN.md).  Every numerical step is a kernel: the operator application (api.cu), the
// subspace matrices V^T W and the Ritz/residual combinations on the FP64 tensor cores (gemm.cu), the small
// dense eigenproblem by parallel-order cyclic Jacobi in one CTA, the preconditioner, Gram-Schmidt and P_c.
// The host only decides convergence from the residual norms.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <vector>
#include "ctx.h"

using namespace tddft;

namespace {

// ---- small symmetric eigenproblem: parallel-order cyclic Jacobi, one CTA ---------------------------------
// H [m][m] row-major (destroyed), Y [m][m] receives eigenvectors as columns, evals ascending.
__global__ void __launch_bounds__(512) jacobi_eigh_kernel(double* __restrict__ H, double* __restrict__ Y, int m,
                                                         double* __restrict__ evals, double* __restrict__ Ysorted) {
    extern __shared__ double sh[];
    const int mp = (m + 1) & ~1;            // even number of players; index m (if odd) is a bye
    const int np = mp / 2;
    double* cs = sh;                          // [np][2]
    int* pq = (int*)(sh + 2 * np);            // [np][2]
    __shared__ double s_off, s_tot;
    const int tid = threadIdx.x, nt = blockDim.x;
    for (int i = tid; i < m * m; i += nt) Y[i] = (i / m == i % m) ? 1.0 : 0.0;
    __syncthreads();
    for (int sweep = 0; sweep < 40; ++sweep) {
        // convergence: off-diagonal Frobenius norm against the total
        if (tid == 0) { s_off = 0.0; s_tot = 0.0; }
        __syncthreads();
        double off = 0.0, tot = 0.0;
        for (int i = tid; i < m * m; i += nt) { const double v = H[i]; tot += v * v; if (i / m != i % m) off += v * v; }
        atomicAdd(&s_off, off); atomicAdd(&s_tot, tot);
        __syncthreads();
        if (s_off <= 1e-30 * s_tot || s_tot == 0.0) break;
        __syncthreads();
        for (int round = 0; round < mp - 1; ++round) {
            for (int i = tid; i < np; i += nt) {
                int a, b;
                if (i == 0) { a = mp - 1; b = round; }
                else { a = (round + i) % (mp - 1); b = (round + mp - 1 - i) % (mp - 1); }
                int p = min(a, b), q = max(a, b);
                double c = 1.0, s = 0.0;
                if (q < m) {
                    const double apq = H[p * m + q];
                    if (apq != 0.0) {
                        const double theta = (H[q * m + q] - H[p * m + p]) / (2.0 * apq);
                        const double t = (theta >= 0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                        c = 1.0 / sqrt(t * t + 1.0); s = t * c;
                    }
                } else { p = -1; }
                pq[2 * i] = p; pq[2 * i + 1] = q; cs[2 * i] = c; cs[2 * i + 1] = s;
            }
            __syncthreads();
            for (int w = tid; w < np * m; w += nt) {          // rows: A <- J^T A
                const int i = w / m, k = w - i * m, p = pq[2 * i], q = pq[2 * i + 1];
                if (p < 0) continue;
                const double c = cs[2 * i], s = cs[2 * i + 1];
                const double ap = H[p * m + k], aq = H[q * m + k];
                H[p * m + k] = c * ap - s * aq; H[q * m + k] = s * ap + c * aq;
            }
            __syncthreads();
            for (int w = tid; w < np * m; w += nt) {          // columns: A <- A J, Y <- Y J
                const int i = w / m, k = w - i * m, p = pq[2 * i], q = pq[2 * i + 1];
                if (p < 0) continue;
                const double c = cs[2 * i], s = cs[2 * i + 1];
                const double ap = H[k * m + p], aq = H[k * m + q];
                H[k * m + p] = c * ap - s * aq; H[k * m + q] = s * ap + c * aq;
                const double yp = Y[k * m + p], yq = Y[k * m + q];
                Y[k * m + p] = c * yp - s * yq; Y[k * m + q] = s * yp + c * yq;
            }
            __syncthreads();
        }
    }
    __syncthreads();
    // ascending order: rank of each eigenvalue (ties broken by index), then permuted copy
    for (int i = tid; i < m; i += nt) {
        const double e = H[i * m + i];
        int rank = 0;
        for (int j = 0; j < m; ++j) { const double f = H[j * m + j]; if (f < e || (f == e && j < i)) ++rank; }
        evals[rank] = e;
        for (int k = 0; k < m; ++k) Ysorted[k * m + rank] = Y[k * m + i];
    }
}

// t = r / d, d = |G|^2/2 - eps_v - theta, |d| floored at 1e-2 keeping its sign (reading A11)
struct PrecBlocks { long off[2]; int nocc[2]; const double* eig[2]; int nblocks; };
__global__ void precondition_kernel(const cplx* __restrict__ r, cplx* __restrict__ t, long L, long npwh, PrecBlocks pb,
                                    const double* __restrict__ kin, const double* __restrict__ theta, int root) {
    const double th = theta[root];
    for (long e = blockIdx.x * (long)blockDim.x + threadIdx.x; e < L; e += (long)gridDim.x * blockDim.x) {
        const int b = (pb.nblocks == 2 && e >= pb.off[1]) ? 1 : 0;
        const long le = e - pb.off[b];
        const long v = le / npwh, g = le - v * npwh;
        double d = kin[g] - pb.eig[b][v] - th;
        if (fabs(d) < 1e-2) d = d < 0 ? -1e-2 : 1e-2;
        const cplx x = r[e];
        t[e] = make_double2(x.x / d, x.y / d);
    }
}
__global__ void scale_kernel(double* __restrict__ x, long n, const double* __restrict__ norm2, double* __restrict__ dst) {
    const double s = 1.0 / sqrt(norm2[0]);
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) dst[i] = x[i] * s;
}
// r_i <- r_i - theta_i x_i for the first nroots rows
__global__ void residual_kernel(double* __restrict__ R, const double* __restrict__ X, long n, const double* __restrict__ theta) {
    const double th = theta[blockIdx.y];
    double* r = R + (long)blockIdx.y * n; const double* x = X + (long)blockIdx.y * n;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) r[i] = fma(-th, x[i], r[i]);
}
__global__ void symmetrize_kernel(double* __restrict__ H, int m) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m * m) return;
    const int r = i / m, c = i % m;
    if (r < c) { const double v = 0.5 * (H[r * m + c] + H[c * m + r]); H[r * m + c] = v; H[c * m + r] = v; }
}
// ---- projector-aware correction (reading A11b of DESIGN.md) ----------------------------------------------------------------
// For every function v of a spin block and Ritz value theta: solve P_c (T - lambda_v) P_c t = r on range(P_c), lambda_v = eps_v + theta:
//   t = M^-1 (r - Phi c),  c = S^-1 Phi^T M^-1 r,  S = Phi^T M^-1 Phi,  M = diag(|G|^2/2 - lambda_v) with |M| floored at 1e-2 (sign kept).
constexpr double kDenFloor = 1e-2;
__device__ __forceinline__ double pc_den(double kin, double lam) {
    double d = kin - lam;
    if (fabs(d) < kDenFloor) d = d < 0 ? -kDenFloor : kDenFloor;
    return d;
}
__global__ void pc_lambda_kernel(const double* __restrict__ eig, const double* __restrict__ theta, int root, int n, double* __restrict__ lam) {
    const int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v < n) lam[v] = eig[v] + theta[root];
}
// weighted != 0: out[v][k] = gamma_k in[v][k] / d_v(k) (gamma: the Gamma inner-product weights 2, 1 for Re c(0), 0 for Im c(0));
// weighted == 0: out[v][k] = in[v][k] / d_v(k)
__global__ void pc_divide_kernel(const double* __restrict__ in, double* __restrict__ out, long k2, const double* __restrict__ kin,
                                 const double* __restrict__ lam, int weighted) {
    const int v = blockIdx.y;
    const double l = lam[v];
    const double* src = in + (long)v * k2; double* dst = out + (long)v * k2;
    for (long k = blockIdx.x * (long)blockDim.x + threadIdx.x; k < k2; k += (long)gridDim.x * blockDim.x) {
        const double d = pc_den(kin[k >> 1], l);
        double w = 1.0 / d;
        if (weighted) w = (k >= 2) ? 2.0 / d : (k == 0 ? 1.0 / d : 0.0);
        dst[k] = src[k] * w;
    }
}
__global__ void fill_kernel(double* __restrict__ x, int n, double v) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) x[i] = v;
}
// w[row][k] = kin[k/2] x[row][k]: the kinetic operator on half-sphere functions stored as 2 npwh reals
__global__ void kin_mul_kernel(const double* __restrict__ x, double* __restrict__ w, long k2, const double* __restrict__ kin) {
    const double* src = x + (long)blockIdx.y * k2; double* dst = w + (long)blockIdx.y * k2;
    for (long k = blockIdx.x * (long)blockDim.x + threadIdx.x; k < k2; k += (long)gridDim.x * blockDim.x) dst[k] = kin[k >> 1] * src[k];
}
__global__ void unit_kernel(double* __restrict__ x, long k2, long idx) {
    for (long k = blockIdx.x * (long)blockDim.x + threadIdx.x; k < k2; k += (long)gridDim.x * blockDim.x) x[k] = k == idx ? 1.0 : 0.0;
}
// One CTA solves one dense system S x = b by Gaussian elimination with partial pivoting (S is symmetric but indefinite: M has both
// signs), right-hand side carried along in shared memory.  S [nsys][n][n] is destroyed.  The solution leaves negated and
// transposed: CT[u][v0 + sys] = -x[u], the operand of the GEMM  t = r - sum_u c_u phi_u.
__global__ void __launch_bounds__(512) lu_solve_kernel(double* __restrict__ Sall, const double* __restrict__ Ball, double* __restrict__ CT,
                                                      int ldct, int n, int v0) {
    extern __shared__ double sh[];
    double* prow = sh; double* lcol = sh + n; double* x = sh + 2 * n;
    __shared__ double redv[16]; __shared__ int redi[16]; __shared__ int piv;
    double* A = Sall + (size_t)blockIdx.x * n * n;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nw = blockDim.x >> 5;
    for (int i = tid; i < n; i += blockDim.x) x[i] = Ball[(size_t)blockIdx.x * n + i];
    __syncthreads();
    for (int k = 0; k < n; ++k) {
        double bv = -1.0; int bi = k;
        for (int i = k + tid; i < n; i += blockDim.x) { const double a = fabs(A[(size_t)i * n + k]); if (a > bv) { bv = a; bi = i; } }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_down_sync(0xffffffffu, bv, o); const int oi = __shfl_down_sync(0xffffffffu, bi, o);
            if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
        }
        if (lane == 0) { redv[warp] = bv; redi[warp] = bi; }
        __syncthreads();
        if (tid == 0) {
            double b = redv[0]; int p = redi[0];
            for (int w = 1; w < nw; ++w) if (redv[w] > b || (redv[w] == b && redi[w] < p)) { b = redv[w]; p = redi[w]; }
            piv = p;
        }
        __syncthreads();
        const int p = piv;
        if (p != k) {
            for (int j = k + tid; j < n; j += blockDim.x) { const double a = A[(size_t)k * n + j]; A[(size_t)k * n + j] = A[(size_t)p * n + j]; A[(size_t)p * n + j] = a; }
            if (tid == 0) { const double a = x[k]; x[k] = x[p]; x[p] = a; }
            __syncthreads();
        }
        for (int j = k + tid; j < n; j += blockDim.x) prow[j] = A[(size_t)k * n + j];
        __syncthreads();
        double pv = prow[k];
        if (fabs(pv) < 1e-300) pv = 1e-300;          // exactly singular S (lambda on the spectrum of P_c T P_c): regularised
        for (int i = k + 1 + tid; i < n; i += blockDim.x) lcol[i] = A[(size_t)i * n + k] / pv;
        __syncthreads();
        const double xk = x[k];
        for (int i = k + 1 + warp; i < n; i += nw) {
            const double l = lcol[i];
            double* row = A + (size_t)i * n;
            for (int j = k + 1 + lane; j < n; j += 32) row[j] = fma(-l, prow[j], row[j]);
            if (lane == 0) x[i] = fma(-l, xk, x[i]);
        }
        __syncthreads();
    }
    for (int k = n - 1; k >= 0; --k) {
        if (tid == 0) { double pv = A[(size_t)k * n + k]; if (fabs(pv) < 1e-300) pv = 1e-300; x[k] /= pv; }
        __syncthreads();
        const double xk = x[k];
        for (int i = tid; i < k; i += blockDim.x) x[i] = fma(-A[(size_t)i * n + k], xk, x[i]);
        __syncthreads();
    }
    for (int i = tid; i < n; i += blockDim.x) CT[(size_t)i * ldct + v0 + blockIdx.x] = -x[i];
}

}  // namespace

namespace tddft {
struct Blk { int src, tgt; long off; };
}

#define DV_CUDA(call) TD_CUDA(c, call)

extern "C" __attribute__((visibility("default")))
int tddft_davidson(tddft_ctx* c, int nroots, int mode, double* evals, double* evecs, int* iters, double* resnorms) {
    if (!c) return TDDFT_EINVAL;
    if (!evals || nroots < 1 || mode < 0 || mode > 2) return set_err(c, TDDFT_EINVAL, "davidson: bad argument");
    const long L = vector_len(c, mode);
    if (L < 0) return set_err(c, TDDFT_EINVAL, "spin flip needs nspin = 2");
    if (c->shard_count > 1) return set_err(c, TDDFT_EINVAL, "davidson: not available on a sharded context (its applies would be partial sums)");
    TD_CUDA(c, cudaSetDevice(c->device));
    const long n2 = 2 * L, npwh = c->hp.npwh;
    cudaStream_t st = c->stream;
    const int max_sub = c->dav_max_subspace > 0 ? c->dav_max_subspace : 12 * nroots;
    const int max_iter = c->dav_max_iter > 0 ? c->dav_max_iter : 200;
    const double tol = c->dav_tol > 0 ? c->dav_tol : 1e-6;
    const int nstart = (c->dav_x0 && c->dav_nx0 > 0) ? c->dav_nx0 : 2 * nroots;
    if (max_sub < std::max(2 * nroots, nstart)) return set_err(c, TDDFT_EINVAL, "davidson: max_subspace must be >= max(2*nroots, n_x0)");
    // blocks of the vector layout
    std::vector<Blk> blocks;
    if (mode == TDDFT_SPIN_CONSERVING) { long off = 0; for (int s = 0; s < c->nspin; ++s) { blocks.push_back({s, s, off}); off += (long)c->nocc[s] * npwh; } }
    else { const int src = mode == TDDFT_SPIN_FLIP ? 0 : 1; blocks.push_back({src, 1 - src, 0}); }
    PrecBlocks pb{}; pb.nblocks = (int)blocks.size();
    int maxocc = 0;
    for (size_t b = 0; b < blocks.size(); ++b) { pb.off[b] = blocks[b].off; pb.nocc[b] = c->nocc[blocks[b].src]; pb.eig[b] = c->d_eig[blocks[b].src]; maxocc = std::max(maxocc, std::max(c->nocc[blocks[b].src], c->nocc[blocks[b].tgt])); }

    // ---- buffers ----------------------------------------------------------------------------------
    double *V = nullptr, *W = nullptr, *XR = nullptr, *T = nullptr, *small = nullptr, *Oproj = nullptr;
    const int splits = (int)std::max<long>(1, std::min<long>(256, n2 / 65536));
    const size_t small_n = (size_t)max_sub * max_sub * (3 + splits) + 4 * max_sub + 64;
    double *pcS = nullptr, *pcRS = nullptr, *pcB = nullptr, *pcLam = nullptr, *fbuf_owner = nullptr, *Ufun = nullptr;
    auto cleanup = [&]() { cudaFree(fbuf_owner); cudaFree(Ufun); cudaFree(V); cudaFree(W); cudaFree(XR); cudaFree(T); cudaFree(small); cudaFree(Oproj); cudaFree(pcS); cudaFree(pcRS); cudaFree(pcB); cudaFree(pcLam); cudaGetLastError(); };
#define DV_TRY(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { cleanup(); return set_err(c, e_ == cudaErrorMemoryAllocation ? TDDFT_ENOMEM : TDDFT_ECUDA, std::string("davidson: " #call ": ") + cudaGetErrorString(e_)); } } while (0)
#define DV_RC(expr) do { int rc_ = (expr); if (rc_) { cleanup(); return rc_; } } while (0)
    DV_TRY(cudaMalloc((void**)&V, sizeof(double) * n2 * max_sub));
    DV_TRY(cudaMalloc((void**)&W, sizeof(double) * n2 * max_sub));
    DV_TRY(cudaMalloc((void**)&XR, sizeof(double) * n2 * 3 * nroots));     // X (Ritz), R (residual / W-combination), WY for restarts
    DV_TRY(cudaMalloc((void**)&T, sizeof(double) * n2));
    DV_TRY(cudaMalloc((void**)&small, sizeof(double) * small_n));
    const size_t oproj_cap = project_scratch_doubles(c, maxocc, std::max(maxocc, 16), (size_t)1 << 34);
    DV_TRY(cudaMalloc((void**)&Oproj, sizeof(double) * oproj_cap));
    double* X = XR; double* R = XR + n2 * nroots; double* WY = XR + 2 * n2 * nroots;
    double* H = small; double* Hwork = H + (size_t)max_sub * max_sub; double* Y = Hwork + (size_t)max_sub * max_sub;
    double* part = Y + (size_t)max_sub * max_sub; double* theta = part + (size_t)max_sub * max_sub * splits;
    double* coef = theta + max_sub; double* nrm = coef + 2 * max_sub;   // nrm: scratch scalars
    const long wper = 2 * npwh;
    const unsigned eb = (unsigned)std::min<long>(4096, (n2 + 255) / 256);
    long launches = 0;

    auto project_vec = [&](double* x) -> int {     // P_c block by block on one full vector
        for (auto& b : blocks) {
            int rc = project_rows(c, b.tgt, x + 2 * b.off, c->nocc[b.src], c->nocc[b.src], 0, Oproj, oproj_cap);
            if (rc) return rc;
        }
        return TDDFT_OK;
    };
    auto norm2_to_host = [&](const double* x, double* out) -> int {   // Gamma inner product <x|x>
        TD_CUDA(c, launch_gemm_nt(x, n2, x, n2, 1, 0, nrm, 1, 1, 1, n2, wper, 2.0, splits, part, st));
        TD_CUDA(c, cudaMemcpyAsync(out, nrm, sizeof(double), cudaMemcpyDeviceToHost, st));
        TD_CUDA(c, cudaStreamSynchronize(st));
        launches += 2;
        return TDDFT_OK;
    };
    // two passes of classical Gram-Schmidt of t against V[0..m), then P_c again; returns the remaining norm
    auto gs2 = [&](double* t, int m, double* norm_out) -> int {
        for (int pass = 0; pass < 2 && m > 0; ++pass) {
            TD_CUDA(c, launch_gemm_nt(V, n2, t, n2, 1, 0, coef, 1, m, 1, n2, wper, 2.0, splits, part, st));
            TD_CUDA(c, launch_gemm_tn_acc(coef, 1, V, n2, t, n2, 1, 0, 1, n2, m, -1.0, st));
            launches += 3;
        }
        int rc = project_vec(t); if (rc) return rc;
        double n2h = 0; rc = norm2_to_host(t, &n2h); if (rc) return rc;
        *norm_out = std::sqrt(std::max(n2h, 0.0));
        return TDDFT_OK;
    };
    auto append = [&](double* t, int& m) -> int {     // V[m] = t / ||t||  (norm^2 already in nrm[0])
        scale_kernel<<<eb, 256, 0, st>>>(t, n2, nrm, V + (long)m * n2);
        TD_CUDA(c, cudaGetLastError()); ++launches; ++m;
        return TDDFT_OK;
    };

    // projector-aware correction (reading A11b): rows t_v with P_c (T_kin - lam_v) P_c t_v = r_v for n functions of target spin tgt
    const bool pc_aware = c->dav_precond == 0;
    constexpr int PF = 4;                     // conduction functions per spin of the start-vector phase (reading A11c)
    constexpr int FMAX = 8 * PF;
    double* pcCT = nullptr;
    int pc_chunk = 0;
    {
        int maxn = PF, maxt = 0;
        for (auto& b : blocks) { maxn = std::max(maxn, c->nocc[b.src]); maxt = std::max(maxt, c->nocc[b.tgt]); }
        const size_t per = sizeof(double) * (size_t)maxt * maxt;
        pc_chunk = (int)std::max<size_t>(1, std::min<size_t>((size_t)maxn, ((size_t)2 << 30) / per));
        DV_TRY(cudaMalloc((void**)&pcS, std::max(per * pc_chunk, sizeof(double) * 12 * (size_t)maxn * maxt)));   // also the k-split scratch of the rhs GEMM
        DV_TRY(cudaMalloc((void**)&pcRS, sizeof(double) * (size_t)maxn * 2 * npwh));
        DV_TRY(cudaMalloc((void**)&pcB, sizeof(double) * (size_t)maxn * maxt * 2));
        DV_TRY(cudaMalloc((void**)&pcLam, sizeof(double) * maxn));
        pcCT = pcB + (size_t)maxn * maxt;
        cudaFuncSetAttribute(lu_solve_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(double) * 3 * maxt));
    }
    auto solve_rows = [&](const double* rblk, double* tblk, int n, int tgt) -> int {      // shifts lam_v in pcLam[0..n)
        const long k2 = 2 * npwh;
        const int nt = c->nocc[tgt];
        pc_divide_kernel<<<dim3(64, n), 256, 0, st>>>(rblk, pcRS, k2, c->d_kin, pcLam, 1);
        TD_CUDA(c, cudaGetLastError());
        // B[v][u] = <phi_u| M_v^-1 |r_v>
        TD_CUDA(c, launch_gemm_nt(pcRS, k2, c->psi[tgt], k2, nt, 0, pcB, nt, n, nt, k2, 0, 1.0, 12, pcS, st));    // pcS doubles as the k-split scratch
        for (int v0 = 0; v0 < n; v0 += pc_chunk) {
            const int nv = std::min(pc_chunk, n - v0);
            TD_CUDA(c, launch_gram_shift(c->psi[tgt], k2, nt, k2, c->d_kin, pcLam + v0, nv, kDenFloor, pcS, st));
            lu_solve_kernel<<<nv, 512, sizeof(double) * 3 * nt, st>>>(pcS, pcB + (size_t)v0 * nt, pcCT, n, nt, v0);
            TD_CUDA(c, cudaGetLastError());
            launches += 2;
        }
        // t_v = M_v^-1 (r_v - sum_u c_v[u] phi_u)
        if (tblk != rblk) TD_CUDA(c, cudaMemcpyAsync(tblk, rblk, sizeof(double) * (size_t)n * k2, cudaMemcpyDeviceToDevice, st));
        TD_CUDA(c, launch_gemm_tn_acc(pcCT, n, c->psi[tgt], k2, tblk, k2, n, 0, n, k2, nt, 1.0, st));
        pc_divide_kernel<<<dim3(64, n), 256, 0, st>>>(tblk, tblk, k2, c->d_kin, pcLam, 0);
        TD_CUDA(c, cudaGetLastError());
        launches += 5;
        return TDDFT_OK;
    };
    auto precond_projector = [&](int root) -> int {      // T <- correction of root `root`, lam_v = eps_v + theta_root
        for (auto& b : blocks) {
            const int n = c->nocc[b.src];
            pc_lambda_kernel<<<(n + 127) / 128, 128, 0, st>>>(c->d_eig[b.src], theta, root, n, pcLam);
            int rc = solve_rows(R + (long)root * n2 + 2 * b.off, T + 2 * b.off, n, b.tgt); if (rc) return rc;
        }
        return TDDFT_OK;
    };

    // Start-vector phase (reading A11c of DESIGN.md): the PF lowest eigenfunctions u_m (eigenvalues mu_m) of P_c T P_c of one target
    // spin, by a block Davidson in the space of single functions whose correction is the exact inverse at a fixed shift below the
    // spectrum, t = (P_c (T - sigma) P_c)^-1 r with sigma = -0.05 Ha < 0 <= T (a positive definite solve: robust from any start).
    // The eigenvectors of D alone (Eq. 3) are u_m (x) e_v with eigenvalue mu_m - eps_v; the lowest of them start the solver.
    double*& fbuf = fbuf_owner;
    auto conduction_functions = [&](int tgt, double* Uout, double* mu_host) -> int {
        const long k2 = 2 * npwh;
        const int fsplits = (int)std::max<long>(1, std::min<long>(64, k2 / 4096));
        if (!fbuf) TD_CUDA(c, cudaMalloc((void**)&fbuf, sizeof(double) * ((size_t)(2 * FMAX + 3 * PF) * k2 + (size_t)FMAX * FMAX * (3 + fsplits) + 4 * FMAX + 64)));
        double* FV = fbuf; double* FW = FV + (size_t)FMAX * k2; double* FX = FW + (size_t)FMAX * k2; double* FR = FX + (size_t)PF * k2;
        double* FT = FR + (size_t)PF * k2; double* fH = FT + (size_t)PF * k2; double* fHw = fH + FMAX * FMAX; double* fY = fHw + FMAX * FMAX;
        double* fpart = fY + FMAX * FMAX; double* ftheta = fpart + (size_t)FMAX * FMAX * fsplits; double* fcoef = ftheta + FMAX; double* fnrm = fcoef + 2 * FMAX;
        const unsigned fb = (unsigned)std::min<long>(1024, (k2 + 255) / 256);
        const size_t ocap = oproj_cap;
        int fm = 0, fw = 0;
        auto fproject = [&](double* x, int rows) { return project_rows(c, tgt, x, rows, rows, 0, Oproj, ocap); };
        auto fgs_append = [&](double* t) -> int {      // two Gram-Schmidt passes against FV[0..fm), P_c, normalise, append
            for (int pass = 0; pass < 2 && fm > 0; ++pass) {
                TD_CUDA(c, launch_gemm_nt(FV, k2, t, k2, 1, 0, fcoef, 1, fm, 1, k2, k2, 2.0, fsplits, fpart, st));
                TD_CUDA(c, launch_gemm_tn_acc(fcoef, 1, FV, k2, t, k2, 1, 0, 1, k2, fm, -1.0, st));
            }
            int rc = fproject(t, 1); if (rc) return rc;
            TD_CUDA(c, launch_gemm_nt(t, k2, t, k2, 1, 0, fnrm, 1, 1, 1, k2, k2, 2.0, fsplits, fpart, st));
            double q = 0; TD_CUDA(c, cudaMemcpyAsync(&q, fnrm, sizeof(double), cudaMemcpyDeviceToHost, st)); TD_CUDA(c, cudaStreamSynchronize(st));
            if (q > 1e-20) { scale_kernel<<<fb, 256, 0, st>>>(t, k2, fnrm, FV + (size_t)fm * k2); TD_CUDA(c, cudaGetLastError()); ++fm; }
            return TDDFT_OK;
        };
        for (int i = 0; i < PF && i + 1 < k2; ++i) {      // unit vectors on the lowest kinetic energies (real coordinates 0, 2, 3, 4, ...)
            unit_kernel<<<fb, 256, 0, st>>>(FT, k2, i == 0 ? 0 : i + 1);
            int rc = fproject(FT, 1); if (rc) return rc;
            rc = fgs_append(FT); if (rc) return rc;
        }
        if (fm == 0) return set_err(c, TDDFT_EINVAL, "davidson: no conduction function found");
        std::vector<double> hth(FMAX), hr2(PF * PF);
        int np = 0;
        for (int fit = 0; fit < 80; ++fit) {
            if (fw < fm) {      // W = P_c T V on the new rows
                kin_mul_kernel<<<dim3(fb, fm - fw), 256, 0, st>>>(FV + (size_t)fw * k2, FW + (size_t)fw * k2, k2, c->d_kin);
                int rc = fproject(FW + (size_t)fw * k2, fm - fw); if (rc) return rc;
                fw = fm;
            }
            TD_CUDA(c, launch_gemm_nt(FV, k2, FW, k2, fm, 0, fH, fm, fm, fm, k2, k2, 2.0, fsplits, fpart, st));
            symmetrize_kernel<<<(fm * fm + 255) / 256, 256, 0, st>>>(fH, fm);
            TD_CUDA(c, cudaMemcpyAsync(fHw, fH, sizeof(double) * fm * fm, cudaMemcpyDeviceToDevice, st));
            { const int mp = (fm + 1) & ~1; jacobi_eigh_kernel<<<1, 512, sizeof(double) * mp + sizeof(int) * mp, st>>>(fHw, fH, fm, ftheta, fY); }
            np = std::min(PF, fm);
            TD_CUDA(c, cudaMemsetAsync(FX, 0, sizeof(double) * k2 * np, st));
            TD_CUDA(c, cudaMemsetAsync(FR, 0, sizeof(double) * k2 * np, st));
            TD_CUDA(c, launch_gemm_tn_acc(fY, fm, FV, k2, FX, k2, np, 0, np, k2, fm, 1.0, st));
            TD_CUDA(c, launch_gemm_tn_acc(fY, fm, FW, k2, FR, k2, np, 0, np, k2, fm, 1.0, st));
            residual_kernel<<<dim3(fb, np), 256, 0, st>>>(FR, FX, k2, ftheta);
            TD_CUDA(c, launch_gemm_nt(FR, k2, FR, k2, np, 0, fHw, np, np, np, k2, k2, 2.0, fsplits, fpart, st));
            TD_CUDA(c, cudaMemcpyAsync(hth.data(), ftheta, sizeof(double) * fm, cudaMemcpyDeviceToHost, st));
            TD_CUDA(c, cudaMemcpyAsync(hr2.data(), fHw, sizeof(double) * np * np, cudaMemcpyDeviceToHost, st));
            TD_CUDA(c, cudaStreamSynchronize(st));
            bool all = np == PF || np == fm;
            int nnew = 0;
            for (int i = 0; i < np; ++i) if (std::sqrt(std::max(hr2[(size_t)i * np + i], 0.0)) > 1e-7) { all = false; ++nnew; }
            if (c->verbose) { fprintf(stderr, "davidson start phase spin %d it %d m %d mu", tgt, fit, fm); for (int i = 0; i < np; ++i) fprintf(stderr, " %.6e (%.1e)", hth[i], std::sqrt(std::max(hr2[(size_t)i * np + i], 0.0))); fprintf(stderr, "\n"); }
            if (all) break;
            if (fm + nnew > FMAX) {      // restart from the Ritz functions
                TD_CUDA(c, cudaMemsetAsync(FT, 0, sizeof(double) * k2 * np, st));
                TD_CUDA(c, launch_gemm_tn_acc(fY, fm, FW, k2, FT, k2, np, 0, np, k2, fm, 1.0, st));
                TD_CUDA(c, cudaMemcpyAsync(FV, FX, sizeof(double) * k2 * np, cudaMemcpyDeviceToDevice, st));
                TD_CUDA(c, cudaMemcpyAsync(FW, FT, sizeof(double) * k2 * np, cudaMemcpyDeviceToDevice, st));
                fm = np; fw = np;
            }
            fill_kernel<<<1, 64, 0, st>>>(pcLam, np, -0.05);
            int rc = solve_rows(FR, FT, np, tgt); if (rc) return rc;
            const int fm0 = fm;
            for (int i = 0; i < np; ++i) {
                if (std::sqrt(std::max(hr2[(size_t)i * np + i], 0.0)) <= 1e-7) continue;
                rc = fproject(FT + (size_t)i * k2, 1); if (rc) return rc;
                rc = fgs_append(FT + (size_t)i * k2); if (rc) return rc;
            }
            if (fm == fm0) break;
        }
        TD_CUDA(c, cudaMemcpyAsync(Uout, FX, sizeof(double) * k2 * np, cudaMemcpyDeviceToDevice, st));
        TD_CUDA(c, cudaStreamSynchronize(st));
        for (int i = 0; i < PF; ++i) mu_host[i] = i < np ? hth[i] : 1e300;
        return TDDFT_OK;
    };

    // ---- start vectors -------------------------------------------------------------------------------
    int m = 0, mw = 0;
    struct Cand { double e; long off; int tgt, fun; };
    std::vector<Cand> cand;
    if (!(c->dav_x0 && c->dav_nx0 > 0)) {
        // lowest eigenvectors of D (reading A11c): u_m (x) e_v over the blocks, ordered by mu_m - eps_v (host index logic only)
        const long k2 = 2 * npwh;
        DV_TRY(cudaMalloc((void**)&Ufun, sizeof(double) * 2 * PF * k2));
        double mu[2][PF]; bool have[2] = {false, false};
        for (auto& b : blocks) {
            if (!have[b.tgt]) { DV_RC(conduction_functions(b.tgt, Ufun + (size_t)b.tgt * PF * k2, mu[b.tgt])); have[b.tgt] = true; }
            for (int f = 0; f < PF; ++f)
                for (int v = 0; v < c->nocc[b.src]; ++v)
                    if (mu[b.tgt][f] < 1e299) cand.push_back({mu[b.tgt][f] - c->eig_h[b.src][v], b.off + (long)v * npwh, b.tgt, f});
        }
        std::sort(cand.begin(), cand.end(), [](const Cand& x, const Cand& y) { return x.e < y.e || (x.e == y.e && x.off < y.off); });
    }
    for (int i = 0; i < nstart; ++i) {
        if (c->dav_x0 && c->dav_nx0 > 0) DV_TRY(cudaMemcpyAsync(T, c->dav_x0 + (long)i * n2, sizeof(double) * n2, cudaMemcpyDeviceToDevice, st));
        else {
            if (i >= (int)cand.size()) break;
            DV_TRY(cudaMemsetAsync(T, 0, sizeof(double) * n2, st));
            DV_TRY(cudaMemcpyAsync(T + 2 * cand[i].off, Ufun + ((size_t)cand[i].tgt * PF + cand[i].fun) * 2 * npwh, sizeof(double) * 2 * npwh, cudaMemcpyDeviceToDevice, st));
        }
        DV_RC(project_vec(T));
        double nr_ = 0; DV_RC(gs2(T, m, &nr_));
        if (nr_ > 1e-10) DV_RC(append(T, m));
    }
    if (m == 0) { cleanup(); return set_err(c, TDDFT_EINVAL, "davidson: start vectors vanish after projection"); }

    std::vector<double> h_theta(max_sub), h_res(nroots, 0.0), h_r2(nroots * nroots);
    const bool trace = c->verbose != 0;      // one line per iteration on stderr
    int it = 0, status = TDDFT_ENOTCONVERGED, nr = 0;
    for (it = 1; it <= max_iter; ++it) {
        if (mw < m) {      // W = A V for the new columns
            DV_RC(apply_liouville_dev(c, V + (long)mw * n2, W + (long)mw * n2, m - mw, mode));
            launches += c->stats.kernel_launches;
            mw = m;
        }
        // Rayleigh-Ritz: H = (V^T W + W^T V)/2, H y = theta y
        DV_TRY(launch_gemm_nt(V, n2, W, n2, m, 0, H, m, m, m, n2, wper, 2.0, splits, part, st));
        symmetrize_kernel<<<(m * m + 255) / 256, 256, 0, st>>>(H, m);
        DV_TRY(cudaMemcpyAsync(Hwork, H, sizeof(double) * m * m, cudaMemcpyDeviceToDevice, st));
        {
            const int mp = (m + 1) & ~1;
            jacobi_eigh_kernel<<<1, 512, sizeof(double) * mp + sizeof(int) * mp, st>>>(Hwork, H /*scratch for unsorted Y*/, m, theta, Y);
            DV_TRY(cudaGetLastError());
        }
        launches += 4;
        nr = std::min(nroots, m);
        // Ritz vectors X_i = sum_j Y[j][i] V_j and R_i = sum_j Y[j][i] W_j - theta_i X_i
        DV_TRY(cudaMemsetAsync(X, 0, sizeof(double) * n2 * nr, st));
        DV_TRY(cudaMemsetAsync(R, 0, sizeof(double) * n2 * nr, st));
        DV_TRY(launch_gemm_tn_acc(Y, m, V, n2, X, n2, nr, 0, nr, n2, m, 1.0, st));
        DV_TRY(launch_gemm_tn_acc(Y, m, W, n2, R, n2, nr, 0, nr, n2, m, 1.0, st));
        residual_kernel<<<dim3(eb, nr), 256, 0, st>>>(R, X, n2, theta);
        DV_TRY(launch_gemm_nt(R, n2, R, n2, nr, 0, Hwork, nr, nr, nr, n2, wper, 2.0, splits, part, st));
        launches += 5;
        DV_TRY(cudaMemcpyAsync(h_theta.data(), theta, sizeof(double) * m, cudaMemcpyDeviceToHost, st));
        DV_TRY(cudaMemcpyAsync(h_r2.data(), Hwork, sizeof(double) * nr * nr, cudaMemcpyDeviceToHost, st));
        DV_TRY(cudaStreamSynchronize(st));
        bool all = (nr == nroots);
        for (int i = 0; i < nr; ++i) { h_res[i] = std::sqrt(std::max(h_r2[(size_t)i * nr + i], 0.0)); if (h_res[i] > tol) all = false; }
        if (trace) {
            fprintf(stderr, "davidson it %d m %d theta", it, m);
            for (int i = 0; i < nr; ++i) fprintf(stderr, " %.6e", h_theta[i]);
            fprintf(stderr, " res");
            for (int i = 0; i < nr; ++i) fprintf(stderr, " %.2e", h_res[i]);
            fprintf(stderr, "\n");
        }
        if (all) { status = TDDFT_OK; break; }
        if (it == max_iter) break;
        // restart when the new vectors would not fit: keep the Ritz vectors and their images
        int nnew = 0; for (int i = 0; i < nr; ++i) if (h_res[i] > tol) ++nnew;
        if (m + nnew > max_sub) {
            DV_TRY(cudaMemsetAsync(WY, 0, sizeof(double) * n2 * nr, st));
            DV_TRY(launch_gemm_tn_acc(Y, m, W, n2, WY, n2, nr, 0, nr, n2, m, 1.0, st));
            DV_TRY(cudaMemcpyAsync(V, X, sizeof(double) * n2 * nr, cudaMemcpyDeviceToDevice, st));
            DV_TRY(cudaMemcpyAsync(W, WY, sizeof(double) * n2 * nr, cudaMemcpyDeviceToDevice, st));
            ++launches;
            m = nr; mw = nr;
        }
        const int m_before = m;
        const int max_new = c->dav_block > 0 ? c->dav_block : nroots;
        for (int i = 0, added = 0; i < nr && added < max_new; ++i) {
            if (h_res[i] <= tol) continue;
            ++added;
            if (pc_aware) DV_RC(precond_projector(i));
            else { precondition_kernel<<<eb, 256, 0, st>>>((const cplx*)(R + (long)i * n2), (cplx*)T, L, npwh, pb, c->d_kin, theta, i); DV_TRY(cudaGetLastError()); ++launches; }
            DV_RC(project_vec(T));
            double n0 = 0, n1 = 0;
            { double q = 0; DV_RC(norm2_to_host(T, &q)); n0 = std::sqrt(std::max(q, 0.0)); }
            DV_RC(gs2(T, m, &n1));
            if (n1 <= 1e-10 * n0) {      // the correction lies in span V: fall back to the plain residual
                DV_TRY(cudaMemcpyAsync(T, R + (long)i * n2, sizeof(double) * n2, cudaMemcpyDeviceToDevice, st));
                DV_RC(project_vec(T));
                n0 = h_res[i];
                DV_RC(gs2(T, m, &n1));
            }
            if (n1 > 1e-10 * n0) DV_RC(append(T, m));
        }
        if (m == m_before) break;   // nothing could be added
    }
    if (it > max_iter) it = max_iter;
    for (int i = 0; i < nroots; ++i) evals[i] = i < nr ? h_theta[i] : NAN;
    if (resnorms) for (int i = 0; i < nroots; ++i) resnorms[i] = i < nr ? h_res[i] : NAN;
    if (iters) *iters = it;
    if (evecs && nr > 0) { cudaMemcpyAsync(evecs, X, sizeof(double) * n2 * nr, cudaMemcpyDeviceToDevice, st); cudaStreamSynchronize(st); }
    c->stats.kernel_launches = launches;
    cleanup();
    if (status == TDDFT_ENOTCONVERGED) return set_err(c, TDDFT_ENOTCONVERGED, "davidson: not converged within max_iter");
    return TDDFT_OK;
}
