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
// counter-based normal numbers (splitmix64 + Box-Muller) for the library's own start vectors
__device__ __forceinline__ unsigned long long splitmix(unsigned long long x) {
    x += 0x9E3779B97F4A7C15ull; x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull; x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}
__global__ void random_start_kernel(cplx* __restrict__ x, long L, long npwh, unsigned long long seed, double amp, long unit_elem) {
    for (long e = blockIdx.x * (long)blockDim.x + threadIdx.x; e < L; e += (long)gridDim.x * blockDim.x) {
        const unsigned long long a = splitmix(seed + 2ull * (unsigned long long)e), b = splitmix(seed + 2ull * (unsigned long long)e + 1ull);
        const double u1 = ((double)(a >> 11) + 0.5) * (1.0 / 9007199254740992.0), u2 = ((double)(b >> 11) + 0.5) * (1.0 / 9007199254740992.0);
        const double rad = amp * sqrt(-2.0 * log(u1));
        double s, c; sincospi(2.0 * u2, &s, &c);
        x[e] = make_double2(rad * c + (e == unit_elem ? 1.0 : 0.0), (e % npwh == 0) ? 0.0 : rad * s);
    }
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
    auto cleanup = [&]() { cudaFree(V); cudaFree(W); cudaFree(XR); cudaFree(T); cudaFree(small); cudaFree(Oproj); cudaGetLastError(); };
#define DV_TRY(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { cleanup(); return set_err(c, e_ == cudaErrorMemoryAllocation ? TDDFT_ENOMEM : TDDFT_ECUDA, std::string("davidson: " #call ": ") + cudaGetErrorString(e_)); } } while (0)
#define DV_RC(expr) do { int rc_ = (expr); if (rc_) { cleanup(); return rc_; } } while (0)
    DV_TRY(cudaMalloc((void**)&V, sizeof(double) * n2 * max_sub));
    DV_TRY(cudaMalloc((void**)&W, sizeof(double) * n2 * max_sub));
    DV_TRY(cudaMalloc((void**)&XR, sizeof(double) * n2 * 3 * nroots));     // X (Ritz), R (residual / W-combination), WY for restarts
    DV_TRY(cudaMalloc((void**)&T, sizeof(double) * n2));
    DV_TRY(cudaMalloc((void**)&small, sizeof(double) * small_n));
    const size_t oproj_cap = project_scratch_doubles(c, maxocc, maxocc, (size_t)1 << 34);
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

    // ---- start vectors -------------------------------------------------------------------------------
    int m = 0, mw = 0;
    std::vector<long> guess;
    if (!(c->dav_x0 && c->dav_nx0 > 0)) {     // host index logic only: the nstart smallest diagonal elements, ties by position
        std::vector<std::pair<double, long>> cand;
        for (auto& b : blocks)
            for (int v = 0; v < c->nocc[b.src]; ++v)
                for (long g = 0; g < std::min<long>(npwh, nstart); ++g)
                    cand.push_back({0.5 * c->hp.g2[g] - c->eig_h[b.src][v], b.off + (long)v * npwh + g});
        std::sort(cand.begin(), cand.end());
        for (int i = 0; i < nstart; ++i) guess.push_back(cand[std::min<size_t>(i, cand.size() - 1)].second);
    }
    for (int i = 0; i < nstart; ++i) {
        if (c->dav_x0 && c->dav_nx0 > 0) DV_TRY(cudaMemcpyAsync(T, c->dav_x0 + (long)i * n2, sizeof(double) * n2, cudaMemcpyDeviceToDevice, st));
        else {   // unit vector on the i-th smallest diagonal element |G|^2/2 - eps_v plus seeded noise of 2-norm ~1e-3 (reading A11):
                 // the amplitude per component scales with 1/sqrt(2L), or the noise would swamp the unit vector at L ~ 10^7
            random_start_kernel<<<eb, 256, 0, st>>>((cplx*)T, L, npwh, c->seed * 0x100000001B3ull + 0x51ED27ull + (unsigned long long)i * (unsigned long long)(2 * L + 2), 1e-3 / sqrt(2.0 * (double)L), guess[i]);
            DV_TRY(cudaGetLastError()); ++launches;
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
        for (int i = 0; i < nr; ++i) {
            if (h_res[i] <= tol) continue;
            precondition_kernel<<<eb, 256, 0, st>>>((const cplx*)(R + (long)i * n2), (cplx*)T, L, npwh, pb, c->d_kin, theta, i);
            DV_TRY(cudaGetLastError()); ++launches;
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
