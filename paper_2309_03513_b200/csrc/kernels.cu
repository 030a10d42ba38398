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
                                      const double* __restrict__ kin, const double* __restrict__ eig, int accumulate) {
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
        if (!X) {      // plain transform to the sphere, no D term (optionally added to what AX holds)
            cplx ya = make_double2(0.5 * scale * (zp.x + zm.x), 0.5 * scale * (zp.y - zm.y));
            cplx yb = make_double2(0.5 * scale * (zp.y + zm.y), -0.5 * scale * (zp.x - zm.x));
            if (accumulate) { const cplx pa = AX[oa + g]; ya.x += pa.x; ya.y += pa.y; if (hb) { const cplx pb = AX[ob + g]; yb.x += pb.x; yb.y += pb.y; } }
            AX[oa + g] = ya;
            if (hb) AX[ob + g] = yb;
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
                                  cudaStream_t st, bool accumulate) {
    dim3 grid((unsigned)((lay.npwh + 255) / 256), (unsigned)batch);
    gather_unpack2_kernel<<<grid, 256, 0, st>>>(work, nr, idx_p, idx_m, f0, nfun, scale, X, AX, lay, kin, eig, accumulate ? 1 : 0);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------
// a is in the chunked layout [nr/32][nocc*kc][32] (common.h); phi and drho are plain [.][nr]
template <int KC>
__global__ void drho_kernel(const double* __restrict__ phi, const double* __restrict__ a, int nocc, int kc, int kk0, long nr,
                            double* __restrict__ drho, int accumulate) {
    const long r = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (r >= nr) return;
    double acc[KC];
#pragma unroll
    for (int q = 0; q < KC; ++q) acc[q] = 0.0;
    const double* ac = a + (r >> CHUNK_LOG) * ((long)nocc * kc * CHUNK) + (r & (CHUNK - 1));
    for (int v = 0; v < nocc; ++v) {
        const double p = phi[(long)v * nr + r];
        const double* av = ac + ((long)v * kc + kk0) * CHUNK;
#pragma unroll
        for (int q = 0; q < KC; ++q) if (kk0 + q < kc) acc[q] = fma(p, av[q * CHUNK], acc[q]);
    }
#pragma unroll
    for (int q = 0; q < KC; ++q) if (kk0 + q < kc) { double* d = drho + (long)(kk0 + q) * nr + r; *d = accumulate ? *d + acc[q] : acc[q]; }
}
cudaError_t launch_drho(const double* phi, const double* a, int nocc, int kc, long nr, double* drho, cudaStream_t st, bool accumulate) {
    const unsigned nb = (unsigned)((nr + 127) / 128);
    for (int kk0 = 0; kk0 < kc; kk0 += 4) drho_kernel<4><<<nb, 128, 0, st>>>(phi, a, nocc, kc, kk0, nr, drho, accumulate ? 1 : 0);
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
                                const double* __restrict__ a, int nocc, int kc, long nr, double* __restrict__ out, long ftot) {
    const long chunk = blockIdx.x;
    const int lane = threadIdx.x & (CHUNK - 1), sub = threadIdx.x / CHUNK, nsub = blockDim.x / CHUNK;
    const long r = chunk * CHUNK + lane;
    const bool live = r < nr;
    const long base = chunk * (ftot * CHUNK) + lane;
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
                            double* out, cudaStream_t st, long ftot) {
    const long nchunks = (nr + CHUNK - 1) / CHUNK;
    if (ftot <= 0) ftot = (long)nocc * kc;
    if (!V && !vloc && ftot == (long)nocc * kc) return cudaMemsetAsync(out, 0, sizeof(double) * nchunks * CHUNK * nocc * kc, st);
    out_init_kernel<<<(unsigned)nchunks, 256, 0, st>>>(phi, V, vloc, a, nocc, kc, nr, out, ftot);
    return cudaGetLastError();
}

// S5 (the exchange contraction of Eq. 6) lives in contract.cu.

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
    const double* tc = tau + (r >> CHUNK_LOG) * ((long)nj * nt * CHUNK) + (r & (CHUNK - 1));
    for (int j = 0; j < nj; ++j) {
        const double m = M[(long)j * nr + r];
        const double* tj = tc + ((long)j * nt + t0) * CHUNK;
#pragma unroll
        for (int q = 0; q < KT; ++q) if (t0 + q < tend) acc[q] = fma(m, tj[q * CHUNK], acc[q]);
    }
    double* oc = out + (r >> CHUNK_LOG) * (ftot * CHUNK) + (r & (CHUNK - 1));
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
