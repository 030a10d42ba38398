// Rows of SURVEY 8(f) that reuse the pair engine with other operand roles, and the FP64 peak probes of the benchmark:
//   tddft_apply_coupling   K2e - K2d, the off-diagonal block of Eq. 1 (Eqs. 5, 7; spin flip S7, S9)
//   tddft_exchange_apply   V_X psi of Eq. 28 and V_X^ACE of Eq. 29
//   build_ace              the ACE orbitals xi of Eq. 30
// All three are the pattern  out_t(r) += scale * sum_j M_j(r) C[A1_x(t,j) A2_y(t,j)](r): pair FFTs through the same fused
// kernels as tau_vv' (api.cu: pair_potentials_dev), followed by a band sum over j (kernels.cu: pattern_reduce).
#include <algorithm>
#include <cmath>
#include <new>
#include "ctx.h"

using namespace tddft;

namespace {

// plain-layout response density: drho[k][r] = sum_v phi[v][r] a[(v*kc + k)][r]
template <int KC>
__global__ void drho_plain_kernel(const double* __restrict__ phi, const double* __restrict__ a, int nocc, int kc, int kk0, long nr,
                                  double* __restrict__ drho) {
    const long r = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (r >= nr) return;
    double acc[KC];
#pragma unroll
    for (int q = 0; q < KC; ++q) acc[q] = 0.0;
    for (int v = 0; v < nocc; ++v) {
        const double p = phi[(long)v * nr + r];
#pragma unroll
        for (int q = 0; q < KC; ++q) if (kk0 + q < kc) acc[q] = fma(p, a[((long)v * kc + kk0 + q) * nr + r], acc[q]);
    }
#pragma unroll
    for (int q = 0; q < KC; ++q) if (kk0 + q < kc) drho[(long)(kk0 + q) * nr + r] = acc[q];
}

// Pair pattern: targets t = 0..nt_total-1 in groups of gt; every target sums over j = 0..nj-1.  pair(t, j) gives the indices into
// A1 and A2; the band sum multiplies by M[j].  out is a chunked batch of ftot functions, target t is function f0 + t*fstep... the
// caller maps targets to functions through fidx(t).
struct Pattern {
    const double* A1; const double* A2; const double* M;
    int nj; long nt_total;
    double scale;
};
template <class PairFn, class FunFn>
int run_pattern(tddft_ctx* c, const Pattern& pt, PairFn pair, FunFn fidx, double* out, long ftot, double* tau, size_t tau_bytes) {
    const long nr = c->hp.nr;
    const size_t grid_b = sizeof(double) * (size_t)chunked_elems(1, nr);
    int gt = (int)std::min<long>(8, pt.nt_total);
    while (gt > 1 && grid_b * (size_t)gt * pt.nj > tau_bytes) --gt;
    if (grid_b * (size_t)gt * pt.nj > tau_bytes) return set_err(c, TDDFT_ENOMEM, "pair pattern: workspace too small for one target");
    // targets whose function indices are an arithmetic progression can share one reduce launch; fidx is checked per group
    const long npairs_total = pt.nt_total * pt.nj;
    std::vector<int2> pairs((size_t)npairs_total); std::vector<int> slots((size_t)npairs_total);
    size_t q = 0;
    for (long t0 = 0; t0 < pt.nt_total; t0 += gt) {
        const int g = (int)std::min<long>(gt, pt.nt_total - t0);
        for (int tl = 0; tl < g; ++tl)
            for (int j = 0; j < pt.nj; ++j) { pairs[q] = pair(t0 + tl, j); slots[q] = j * g + tl; ++q; }
    }
    int2* d_pairs = nullptr; int* d_slots = nullptr;
    if (cudaMalloc((void**)&d_pairs, sizeof(int2) * pairs.size()) != cudaSuccess || cudaMalloc((void**)&d_slots, sizeof(int) * slots.size()) != cudaSuccess) {
        cudaGetLastError(); cudaFree(d_pairs); return set_err(c, TDDFT_ENOMEM, "pair pattern: pair list allocation failed");
    }
    int rc = TDDFT_OK;
    cudaError_t e = cudaMemcpyAsync(d_pairs, pairs.data(), sizeof(int2) * pairs.size(), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_slots, slots.data(), sizeof(int) * slots.size(), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) rc = set_err(c, TDDFT_ECUDA, std::string("pair pattern: ") + cudaGetErrorString(e));
    long off = 0;
    for (long t0 = 0; t0 < pt.nt_total && !rc; t0 += gt) {
        const int g = (int)std::min<long>(gt, pt.nt_total - t0);
        const long np = (long)g * pt.nj;
        { StageTimer tm(c, ST_S4);
          rc = pair_potentials_dev(c, pt.A1, pt.A2, d_pairs + off, d_slots + off, np, 2 * c->fft_batch, tau, 1, np); }
        if (rc) break;
        StageTimer tm(c, ST_S5);
        // one reduce launch per run of targets with a constant function stride
        int tl = 0;
        while (tl < g && !rc) {
            const long f0 = fidx(t0 + tl);
            long step = 1; int run = 1;
            if (tl + 1 < g) { step = fidx(t0 + tl + 1) - f0; run = 2; while (tl + run < g && fidx(t0 + tl + run) - fidx(t0 + tl + run - 1) == step) ++run; }
            if (step <= 0) { step = 1; run = 1; }
            e = launch_pattern_reduce(pt.M, tau, pt.nj, g, tl, run, nr, out, ftot, f0, step, pt.scale, c->stream);
            if (e != cudaSuccess) rc = set_err(c, TDDFT_ECUDA, std::string("pattern_reduce: ") + cudaGetErrorString(e));
            c->stats.kernel_launches += (run + 3) / 4;
            tl += run;
        }
        off += np;
    }
    cudaStreamSynchronize(c->stream);
    cudaFree(d_pairs); cudaFree(d_slots);
    return rc;
}

// ---- FP64 peak probes (bench.py roofline denominators; "measured on the box in the same run") ------------------
__device__ __forceinline__ void dmma_probe(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__global__ void __launch_bounds__(256) dfma_probe_kernel(double* out, int iters) {
    double x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = 1e-3 * threadIdx.x + i;
    const double a = 1.0000001, b = 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = fma(x[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void __launch_bounds__(256) dmma_probe_kernel(double* out, int iters) {
    double cacc[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) { cacc[i][0] = 1e-3 * threadIdx.x + i; cacc[i][1] = 0.5; }
    const double a = 1.0000001, b = 0.24999;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) dmma_probe(cacc[i][0], cacc[i][1], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += cacc[i][0] + cacc[i][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}


// Read-bandwidth probe for the access pattern of the contraction (contract.cu): every CTA streams PIECE-byte pieces at a 256-byte
// stride (256/PIECE CTAs share each 256-byte run, as the CTAs of one chunk do) through a three-deep cp.async ring.
template <int PIECE>
__global__ void __launch_bounds__(128) stream_probe_kernel(const char* __restrict__ src, long rows_per_chunk, int shar, double* __restrict__ out) {
    extern __shared__ char psm[];
    const unsigned s0 = (unsigned)__cvta_generic_to_shared(psm);
    const long chunk = blockIdx.x / shar; const int sub = blockIdx.x % shar;
    const char* base = src + chunk * rows_per_chunk * 256 + sub * PIECE;
    constexpr int TPR = PIECE / 16, RPP = 128 / TPR, ROWS = 32768 / PIECE;
    const int tr = threadIdx.x / TPR, tp = threadIdx.x % TPR;
    int stage = 0;
    for (long r0 = 0; r0 < rows_per_chunk; r0 += ROWS, ++stage) {
        const unsigned sb = s0 + (stage % 3) * 32768;
        for (int r = tr; r < ROWS && r0 + r < rows_per_chunk; r += RPP)
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sb + r * PIECE + tp * 16), "l"(base + (r0 + r) * 256 + tp * 16) : "memory");
        asm volatile("cp.async.commit_group;" ::: "memory");
        asm volatile("cp.async.wait_group 2;" ::: "memory");
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();
    if (threadIdx.x == 0) out[blockIdx.x & 1023] = ((const double*)psm)[0];
}
template <int PIECE>
cudaError_t stream_probe_run(const char* buf, size_t bytes, double* out, cudaStream_t st, double* gbs) {
    const int shar = 256 / PIECE;
    const long rows = 110L * 110L, nchunks = (long)(bytes / (size_t)(rows * 256));
    cudaError_t e = cudaFuncSetAttribute(stream_probe_kernel<PIECE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 98304);
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    stream_probe_kernel<PIECE><<<(unsigned)(nchunks * shar), 128, 98304, st>>>(buf, rows, shar, out);
    cudaEventRecord(e0, st);
    stream_probe_kernel<PIECE><<<(unsigned)(nchunks * shar), 128, 98304, st>>>(buf, rows, shar, out);
    cudaEventRecord(e1, st);
    e = cudaEventSynchronize(e1);
    float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    *gbs = (double)nchunks * rows * 256.0 / (ms * 1e6);
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace

namespace tddft {

// W_i = V_X R_i = - sum_v phi_v C[phi_v R_i] for nfun functions R given in real space (plain [nfun][nr]); result in the sphere,
// rows of W [nfun][npwh] (Eq. 28).  Workspace from the arena.
static int exchange_real_to_sphere(tddft_ctx* c, int spin, const double* R, long nfun, cplx* W) {
    const long nr = c->hp.nr, npwh = c->hp.npwh;
    const int N = c->nocc[spin];
    const size_t grid_b = sizeof(double) * (size_t)chunked_elems(1, nr);
    const size_t budget = workspace_budget(c);
    // chunk of functions whose chunked out batch plus one tau group fits
    long fc = nfun;
    const size_t tau_min = grid_b * (size_t)N;
    while (fc > 1 && grid_b * (size_t)fc + std::min<size_t>(8, (size_t)fc) * tau_min > budget) fc = (fc + 1) / 2;
    const size_t tau_bytes = std::min<size_t>(8, (size_t)fc) * tau_min;
    if (grid_b * (size_t)fc + tau_min > budget) return set_err(c, TDDFT_ENOMEM, "exchange: workspace budget too small");
    TD_RC(ensure_arena(c, grid_b * (size_t)fc + tau_bytes + 512));
    double* out = (double*)c->arena;
    double* tau = (double*)(c->arena + (grid_b * (size_t)fc + 255) / 256 * 256);
    TD_RC(ensure_phi(c, spin));
    const double* phi = c->d_phi[spin];
    for (long f0 = 0; f0 < nfun; f0 += fc) {
        const long nf = std::min(fc, nfun - f0);
        TD_CUDA(c, cudaMemsetAsync(out, 0, grid_b * (size_t)nf, c->stream));
        Pattern pt{R + f0 * nr, phi, phi, N, nf, -1.0};      // A1 = the functions (shared by the two pairs of a packed grid), A2 = M = phi_v
        TD_RC(run_pattern(c, pt, [&](long t, int j) { return make_int2((int)t, j); }, [&](long t) { return t; }, out, nf, tau, tau_bytes));
        FunLayout lay{0, f0 * npwh, npwh, 1, 0};             // row f of W at W + (f0 + f) * npwh
        TD_RC(to_sphere_plus_d(c, out, (int)nf, nullptr, W, lay, nullptr));
    }
    return TDDFT_OK;
}

// xi of Eq. 30: W = V_X [phi_occ; phi_extra], M = Phi^T W = -L L^T, xi = L^-1 W (rows)
int build_ace(tddft_ctx* c, int spin, const double* psi_extra, int n_extra) {
    const long nr = c->hp.nr, npwh = c->hp.npwh, k2 = 2 * npwh;
    const int N = c->nocc[spin], na = N + n_extra;
    if (c->d_U[spin]) return set_err(c, TDDFT_EUNSUPPORTED, "ace together with wannier_u is not supported");
    cplx *orb = nullptr, *W = nullptr; double *R = nullptr, *small = nullptr; int* status = nullptr;
    auto cleanup = [&]() { cudaFree(orb); cudaFree(W); cudaFree(R); cudaFree(small); cudaFree(status); cudaGetLastError(); };
    const int splits = 8;
#define ACE_TRY(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { cleanup(); return set_err(c, e_ == cudaErrorMemoryAllocation ? TDDFT_ENOMEM : TDDFT_ECUDA, std::string("ace: " #call ": ") + cudaGetErrorString(e_)); } } while (0)
#define ACE_RC(expr) do { int rc_ = (expr); if (rc_) { cleanup(); return rc_; } } while (0)
    ACE_TRY(cudaMalloc((void**)&orb, sizeof(cplx) * (size_t)na * npwh));
    ACE_TRY(cudaMalloc((void**)&W, sizeof(cplx) * (size_t)na * npwh));
    ACE_TRY(cudaMalloc((void**)&small, sizeof(double) * (size_t)na * na * (2 + splits)));
    ACE_TRY(cudaMalloc((void**)&status, sizeof(int)));
    ACE_TRY(cudaMemcpyAsync(orb, c->psi[spin], sizeof(cplx) * (size_t)N * npwh, cudaMemcpyDeviceToDevice, c->stream));
    if (n_extra > 0) ACE_TRY(cudaMemcpyAsync(orb + (size_t)N * npwh, psi_extra, sizeof(cplx) * (size_t)n_extra * npwh, cudaMemcpyDeviceToDevice, c->stream));
    // W_i for the occupied orbitals (their real-space form is already there) and for the extra ones
    ACE_RC(ensure_phi(c, spin));
    ACE_RC(exchange_real_to_sphere(c, spin, c->d_phi[spin], N, W));
    if (n_extra > 0) {
        ACE_TRY(cudaMalloc((void**)&R, sizeof(double) * (size_t)n_extra * nr));
        FunLayout lay{0, 0, npwh, 1, 0};
        ACE_RC(to_real_space(c, (const cplx*)psi_extra, lay, n_extra, R, 0));
        ACE_RC(exchange_real_to_sphere(c, spin, R, n_extra, W + (size_t)N * npwh));
    }
    double* Mm = small; double* Linv = small + (size_t)na * na; double* part = Linv + (size_t)na * na;
    ACE_TRY(launch_gemm_nt((const double*)orb, k2, (const double*)W, k2, na, 0, Mm, na, na, na, k2, k2, 2.0, splits, part, c->stream));
    ACE_TRY(launch_symmetrize(Mm, na, -1.0, c->stream));           // -M, symmetrised: positive definite
    ACE_TRY(launch_chol_inv(Mm, Linv, na, status, c->stream));
    int st = 0;
    ACE_TRY(cudaMemcpyAsync(&st, status, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    ACE_TRY(cudaStreamSynchronize(c->stream));
    if (st) { cleanup(); return set_err(c, TDDFT_EINVAL, "ace: -<phi_i|V_X phi_j> is not positive definite (orbitals linearly dependent?)"); }
    // xi_k = sum_i (L^-1)[k][i] W_i : C[m = k][g] += sum_i At[i][k] W[i][g] with At = (L^-1)^T, i.e. At[i][k] = Linv[k][i]
    ACE_TRY(cudaMalloc((void**)&c->d_xi[spin], sizeof(cplx) * (size_t)na * npwh));
    ACE_TRY(cudaMemsetAsync(c->d_xi[spin], 0, sizeof(cplx) * (size_t)na * npwh, c->stream));
    {   // transpose Linv on the host side of the stream: small matrix
        std::vector<double> h((size_t)na * na), ht((size_t)na * na);
        ACE_TRY(cudaMemcpy(h.data(), Linv, sizeof(double) * h.size(), cudaMemcpyDeviceToHost));
        for (int k = 0; k < na; ++k) for (int i = 0; i < na; ++i) ht[(size_t)i * na + k] = h[(size_t)k * na + i];
        ACE_TRY(cudaMemcpy(Mm, ht.data(), sizeof(double) * ht.size(), cudaMemcpyHostToDevice));
    }
    ACE_TRY(launch_gemm_tn_acc(Mm, na, (const double*)W, k2, (double*)c->d_xi[spin], k2, na, 0, na, k2, na, 1.0, c->stream));
    ACE_TRY(cudaStreamSynchronize(c->stream));
    c->n_ace[spin] = na;
    cleanup();
#undef ACE_TRY
#undef ACE_RC
    return TDDFT_OK;
}

}  // namespace tddft

extern "C" {
#pragma GCC visibility push(default)

int tddft_exchange_apply(tddft_ctx* c, int spin, const double* Y, double* VY, long nfun, int use_ace) {
    if (!c || !Y || !VY || nfun < 1 || spin < 0 || spin >= c->nspin || Y == VY) return TDDFT_EINVAL;
    try {
        TD_CUDA(c, cudaSetDevice(c->device));
        const long nr = c->hp.nr, npwh = c->hp.npwh;
        c->stats = tddft_stats{};
        if (use_ace) {
            if (c->n_ace[spin] <= 0) return set_err(c, TDDFT_EINVAL, "exchange_apply: the context holds no ACE operator (options.ace)");
            TD_CUDA(c, cudaMemsetAsync(VY, 0, sizeof(cplx) * (size_t)nfun * npwh, c->stream));
            const size_t cap = project_scratch_doubles(c, c->n_ace[spin], (int)nfun, (size_t)1 << 34);
            TD_RC(ensure_arena(c, sizeof(double) * cap));
            return lowrank_rows(c, (const double*)c->d_xi[spin], c->n_ace[spin], Y, VY, (int)nfun, (int)nfun, 0, -1.0, (double*)c->arena, cap);
        }
        if (c->d_U[spin]) return set_err(c, TDDFT_EUNSUPPORTED, "exchange_apply with wannier_u is not supported");
        double* R = nullptr;
        if (cudaMalloc((void**)&R, sizeof(double) * (size_t)nfun * nr) != cudaSuccess) { cudaGetLastError(); return set_err(c, TDDFT_ENOMEM, "exchange_apply: allocation failed"); }
        FunLayout lay{0, 0, npwh, 1, 0};
        int rc = to_real_space(c, (const cplx*)Y, lay, (int)nfun, R, 0);
        if (!rc) rc = exchange_real_to_sphere(c, spin, R, nfun, (cplx*)VY);
        cudaStreamSynchronize(c->stream);
        cudaFree(R);
        return rc;
    } catch (const std::bad_alloc&) { return set_err(c, TDDFT_ENOMEM, "exchange_apply: host allocation failed"); }
}

int tddft_fp64_peak(tddft_ctx* c, double* dfma_tflops, double* dmma_tflops) {
    if (!c || !dfma_tflops || !dmma_tflops) return TDDFT_EINVAL;
    TD_CUDA(c, cudaSetDevice(c->device));
    const int ctas = 8 * c->num_sms, thr = 256, iters = 20000;
    double* buf = nullptr;
    TD_CUDA(c, cudaMalloc((void**)&buf, sizeof(double) * ctas * thr));
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    float ms = 0;
    double best[2] = {0.0, 0.0};
    for (int rep = 0; rep < 4; ++rep) {      // first repetition is the warm-up
        cudaEventRecord(e0, c->stream);
        dfma_probe_kernel<<<ctas, thr, 0, c->stream>>>(buf, iters);
        cudaEventRecord(e1, c->stream); cudaEventSynchronize(e1); cudaEventElapsedTime(&ms, e0, e1);
        if (rep) best[0] = std::max(best[0], 2.0 * 16 * (double)iters * ctas * thr / (ms * 1e-3) / 1e12);
        cudaEventRecord(e0, c->stream);
        dmma_probe_kernel<<<ctas, thr, 0, c->stream>>>(buf, iters);
        cudaEventRecord(e1, c->stream); cudaEventSynchronize(e1); cudaEventElapsedTime(&ms, e0, e1);
        // one m8n8k4 DMMA = 8*8*4 multiply-adds per warp
        if (rep) best[1] = std::max(best[1], 2.0 * 256 * 8 * (double)iters * ctas * (thr / 32) / (ms * 1e-3) / 1e12);
    }
    cudaError_t e = cudaGetLastError();
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(buf);
    if (e != cudaSuccess) return set_err(c, TDDFT_ECUDA, cudaGetErrorString(e));
    *dfma_tflops = best[0]; *dmma_tflops = best[1];
    return TDDFT_OK;
}

int tddft_stream_probe(tddft_ctx* c, int piece_bytes, double* gbs) {
    if (!c || !gbs || (piece_bytes != 32 && piece_bytes != 64 && piece_bytes != 128 && piece_bytes != 256)) return TDDFT_EINVAL;
    TD_CUDA(c, cudaSetDevice(c->device));
    const size_t bytes = (size_t)8 << 30;                       // well beyond the 126 MB L2
    char* buf = nullptr; bool own = false;
    if (c->arena_bytes >= bytes + 8192) buf = c->arena + 8192;
    else { if (cudaMalloc((void**)&buf, bytes) != cudaSuccess) { cudaGetLastError(); return set_err(c, TDDFT_ENOMEM, "stream probe: allocation failed"); } own = true; cudaMemsetAsync(buf, 0, bytes, c->stream); }
    double* out = nullptr;
    if (cudaMalloc((void**)&out, 8192) != cudaSuccess) { cudaGetLastError(); if (own) cudaFree(buf); return set_err(c, TDDFT_ENOMEM, "stream probe: allocation failed"); }
    cudaError_t e = piece_bytes == 32 ? stream_probe_run<32>(buf, bytes, out, c->stream, gbs)
                  : piece_bytes == 64 ? stream_probe_run<64>(buf, bytes, out, c->stream, gbs)
                  : piece_bytes == 128 ? stream_probe_run<128>(buf, bytes, out, c->stream, gbs)
                                       : stream_probe_run<256>(buf, bytes, out, c->stream, gbs);
    cudaFree(out); if (own) cudaFree(buf);
    if (e != cudaSuccess) return set_err(c, TDDFT_ECUDA, std::string("stream probe: ") + cudaGetErrorString(e));
    return TDDFT_OK;
}

int tddft_apply_coupling(tddft_ctx* c, const double* Xd, double* BXd, int nvec, int mode) {
    if (!c) return TDDFT_EINVAL;
    if (!Xd || !BXd || nvec < 1 || Xd == BXd) return set_err(c, TDDFT_EINVAL, "coupling: bad buffers or nvec < 1");
    if (mode < 0 || mode > 2) return set_err(c, TDDFT_EINVAL, "coupling: unknown mode");
    if (mode != TDDFT_SPIN_CONSERVING && c->nspin != 2) return set_err(c, TDDFT_EINVAL, "spin flip needs nspin = 2");
    if (c->d_U[0] || c->d_U[1]) return set_err(c, TDDFT_EUNSUPPORTED, "coupling with wannier_u is not supported");
    try {
        TD_CUDA(c, cudaSetDevice(c->device));
        const cplx* X = (const cplx*)Xd; cplx* BX = (cplx*)BXd;
        const long nr = c->hp.nr, npwh = c->hp.npwh;
        c->stats = tddft_stats{};
        // blocks of the OUTPUT: functions v over occ(out_occ), living in spin tgt; the input functions v' run over occ(in_occ):
        // spin conserving in_occ = out_occ = tgt = s; spin flip (Eqs. S7, S9): out_occ = s~, tgt = s, in_occ = s (X has the opposite layout)
        struct CB { int out_occ, in_occ, tgt; long off_out, off_in; };
        std::vector<CB> blocks;
        long Lout = 0, Lin = 0;
        if (mode == TDDFT_SPIN_CONSERVING) {
            long off = 0;
            for (int s = 0; s < c->nspin; ++s) { blocks.push_back({s, s, s, off, off}); off += (long)c->nocc[s] * npwh; }
            Lout = Lin = off;
        } else {
            const int so = mode == TDDFT_SPIN_FLIP ? 0 : 1, st = 1 - so;
            blocks.push_back({so, st, st, 0, 0});
            Lout = (long)c->nocc[so] * npwh; Lin = (long)c->nocc[st] * npwh;
        }
        const int nblk = (int)blocks.size();
        const bool hxc = mode == TDDFT_SPIN_CONSERVING && c->use_hartree_fxc;
        const bool sfk = mode != TDDFT_SPIN_CONSERVING && c->sf_xc;
        int maxin = 0, maxout = 0, maxtgt = 0;
        for (auto& b : blocks) { maxin = std::max(maxin, c->nocc[b.in_occ]); maxout = std::max(maxout, c->nocc[b.out_occ]); maxtgt = std::max(maxtgt, c->nocc[b.tgt]); }
        // workspace: a (plain, one block), out (chunked, one block), drho/V/vh, projector scratch, tau (8 targets x nj functions)
        const size_t budget = workspace_budget(c);
        const size_t grid_b = sizeof(double) * (size_t)chunked_elems(1, nr);
        int kc = nvec;
        size_t fixed = 0, tau_bytes = 0;
        for (;;) {
            fixed = grid_b * (size_t)kc * ((size_t)maxin + maxout) + grid_b * (size_t)kc * (2 * nblk + 1)
                  + sizeof(double) * project_scratch_doubles(c, maxtgt, kc * maxout, budget) + 8192;
            tau_bytes = grid_b * 8 * (size_t)maxin;
            if (fixed + tau_bytes <= budget) break;
            if (kc == 1) { tau_bytes = grid_b * (size_t)maxin; if (fixed + tau_bytes <= budget) break; return set_err(c, TDDFT_ENOMEM, "coupling: workspace budget too small"); }
            kc = (kc + 1) / 2;
        }
        TD_RC(ensure_arena(c, fixed + tau_bytes));
        char* p = c->arena;
        auto carve = [&](size_t bytes) { char* q = p; p += (bytes + 255) / 256 * 256; return (double*)q; };
        double* a = carve(grid_b * (size_t)kc * maxin);
        double* out = carve(grid_b * (size_t)kc * maxout);
        std::vector<double*> drho(nblk), V(nblk);
        for (int b = 0; b < nblk; ++b) { drho[b] = carve(grid_b * kc); V[b] = carve(grid_b * kc); }
        double* vh = carve(grid_b * kc);
        const size_t o_cap = project_scratch_doubles(c, maxtgt, kc * maxout, budget);
        double* O = carve(sizeof(double) * o_cap);
        double* tau = carve(tau_bytes);
        c->last_kc = kc; c->last_resident = 0; c->last_pair_tile = 0; c->last_pair_batch = 2 * c->fft_batch;
        const unsigned nbr = (unsigned)((nr + 127) / 128);
        for (int k0 = 0; k0 < nvec; k0 += kc) {
            const int kcc = std::min(kc, nvec - k0);
            auto load = [&](int b) -> int {     // a_(v',k)(r), plain layout [v'*kcc + k][nr]
                StageTimer t(c, ST_S1);
                TD_RC(ensure_phi(c, blocks[b].in_occ));
                FunLayout lay{Lin, blocks[b].off_in, npwh, kcc, k0};
                return to_real_space(c, X, lay, c->nocc[blocks[b].in_occ] * kcc, a, 0);
            };
            int loaded = -1;
            if (hxc || sfk) {
                for (int b = 0; b < nblk; ++b) {
                    TD_RC(load(b)); loaded = b;
                    StageTimer t(c, ST_S23);
                    for (int kk0 = 0; kk0 < kcc; kk0 += 4) drho_plain_kernel<4><<<nbr, 128, 0, c->stream>>>(c->d_phi[blocks[b].in_occ], a, c->nocc[blocks[b].in_occ], kcc, kk0, nr, drho[b]);
                    TD_CUDA(c, cudaGetLastError()); c->stats.kernel_launches += (kcc + 3) / 4;
                }
                StageTimer t(c, ST_S23);
                if (sfk) { TD_CUDA(c, launch_scale_potential(c->d_fsf, drho[0], kcc, nr, V[0], c->stream)); }
                else if (c->nspin == 2) {
                    TD_RC(hartree(c, drho[0], drho[1], 1.0, kcc, vh));
                    TD_CUDA(c, launch_hxc_potential(vh, c->d_fxc[0], drho[0], c->d_fxc[1], drho[1], kcc, nr, V[0], c->stream));
                    TD_CUDA(c, launch_hxc_potential(vh, c->d_fxc[1], drho[0], c->d_fxc[2], drho[1], kcc, nr, V[1], c->stream));
                } else {
                    TD_RC(hartree(c, drho[0], nullptr, 2.0, kcc, vh));
                    TD_CUDA(c, launch_hxc_potential(vh, c->d_fxc[0], drho[0], c->d_fxc[1], drho[0], kcc, nr, V[0], c->stream));
                }
            }
            for (int b = 0; b < nblk; ++b) {
                const CB& bl = blocks[b];
                const int nout = c->nocc[bl.out_occ], nin = c->nocc[bl.in_occ];
                if (loaded != b) { TD_RC(load(b)); loaded = b; }
                // K2e: phi_v V (Eq. 5; with real functions the same potential as K1e)
                TD_RC(ensure_phi(c, bl.out_occ));
                { StageTimer t(c, ST_S5);
                  TD_CUDA(c, launch_out_init(c->d_phi[bl.out_occ], (hxc || sfk) ? V[b] : nullptr, nullptr, nullptr, nout, kcc, nr, out, c->stream)); c->stats.kernel_launches += 1; }
                // K2d (Eq. 7): out_(v,k) -= alpha sum_v' phi_v'(r) C[phi_v a_(v',k)](r): targets t = (k, v), band index j = v'
                if (c->alpha != 0.0) {
                    if (c->phi_shared && bl.out_occ != bl.in_occ) return set_err(c, TDDFT_EUNSUPPORTED, "coupling: spin flip needs both spins' orbitals resident");
                    Pattern pt{c->d_phi[bl.out_occ], a, c->d_phi[bl.in_occ], nin, (long)nout * kcc, -c->alpha};
                    // t = k*nout + v: consecutive targets are consecutive orbitals v of one trial vector (function stride kcc)
                    TD_RC(run_pattern(c, pt,
                        [&](long t, int j) { const int k = (int)(t / nout), v = (int)(t % nout); return make_int2(v, j * kcc + k); },
                        [&](long t) { const long k = t / nout, v = t % nout; return v * kcc + k; }, out, (long)nout * kcc, tau, tau_bytes));
                }
                FunLayout lay{Lout, bl.off_out, npwh, kcc, k0};
                { StageTimer t(c, ST_S6); TD_RC(to_sphere_plus_d(c, out, nout * kcc, nullptr, BX, lay, nullptr)); }
                StageTimer t(c, ST_S8);
                TD_RC(project_rows(c, bl.tgt, (double*)(BX + (long)k0 * Lout + bl.off_out), kcc * nout, nout, 2 * Lout, O, o_cap));
            }
        }
        collect_timing(c);
        return TDDFT_OK;
    } catch (const std::bad_alloc&) { return set_err(c, TDDFT_ENOMEM, "coupling: host allocation failed"); }
}

#pragma GCC visibility pop
}  // extern "C"
