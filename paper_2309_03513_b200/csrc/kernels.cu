// Pointwise, scatter/gather, contraction and LDA kernels of the Liouville hot path (hand-written CUDA, sm_100a).
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
    const double ea = eig[va], eb = hb ? eig[vb] : 0.0;
    const cplx* w = work + (long)b * nr;
    for (long g = blockIdx.x * (long)blockDim.x + threadIdx.x; g < lay.npwh; g += (long)gridDim.x * blockDim.x) {
        const cplx zp = w[idx_p[g]], zm = w[idx_m[g]];
        // c_A = (Z(G) + conj Z(-G))/2,  c_B = (Z(G) - conj Z(-G))/(2i)
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
template <int KC>
__global__ void drho_kernel(const double* __restrict__ phi, const double* __restrict__ a, int nocc, int kc, int kk0, long nr,
                            double* __restrict__ drho) {
    const long r = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (r >= nr) return;
    double acc[KC];
#pragma unroll
    for (int q = 0; q < KC; ++q) acc[q] = 0.0;
    for (int v = 0; v < nocc; ++v) {
        const double p = phi[(long)v * nr + r];
        const double* av = a + ((long)v * kc + kk0) * nr + r;
#pragma unroll
        for (int q = 0; q < KC; ++q) if (kk0 + q < kc) acc[q] = fma(p, av[(long)q * nr], acc[q]);
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

__global__ void out_init_kernel(const double* __restrict__ phi, const double* __restrict__ V, const double* __restrict__ vloc,
                                const double* __restrict__ a, int kc, long nr, double* __restrict__ out) {
    const long r = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (r >= nr) return;
    const int f = blockIdx.y;
    const int v = f / kc, kk = f - v * kc;
    double y = 0.0;
    if (V) y = phi[(long)v * nr + r] * V[(long)kk * nr + r];
    if (vloc) y = fma(vloc[r], a[(long)f * nr + r], y);
    out[(long)f * nr + r] = y;
}
cudaError_t launch_out_init(const double* phi, const double* V, const double* vloc, const double* a, int nocc, int kc, long nr,
                            double* out, cudaStream_t st) {
    if (!V && !vloc) return cudaMemsetAsync(out, 0, sizeof(double) * nr * nocc * kc, st);
    dim3 grid((unsigned)((nr + 255) / 256), (unsigned)(nocc * kc));
    out_init_kernel<<<grid, 256, 0, st>>>(phi, V, vloc, a, kc, nr, out);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------
// S5, first version: one thread per grid point, TI x TK accumulators in registers, FP64 FMA.
template <int TI, int TK>
__global__ void __launch_bounds__(128) contract_kernel(double* __restrict__ out, const double* __restrict__ a, const double* __restrict__ tau,
                                const int* __restrict__ slot, int i0, int ti, int j0, int tj, int kc, long nr, double alpha) {
    const long r = blockIdx.x * (long)blockDim.x + threadIdx.x;
    const int ib = blockIdx.y * TI, kb = blockIdx.z * TK;
    extern __shared__ int sslot[];     // [TI][tj]
    for (int t = threadIdx.x; t < TI * tj; t += blockDim.x) {
        const int i = t / tj, j = t - i * tj;
        sslot[t] = (ib + i < ti) ? slot[(ib + i) * tj + j] : -1;
    }
    __syncthreads();
    if (r >= nr) return;
    double acc[TI][TK];
#pragma unroll
    for (int i = 0; i < TI; ++i)
#pragma unroll
        for (int q = 0; q < TK; ++q) acc[i][q] = 0.0;
    for (int j = 0; j < tj; ++j) {
        double av[TK];
        const double* ap = a + ((long)(j0 + j) * kc + kb) * nr + r;
#pragma unroll
        for (int q = 0; q < TK; ++q) av[q] = (kb + q < kc) ? ap[(long)q * nr] : 0.0;
#pragma unroll
        for (int i = 0; i < TI; ++i) {
            const int s = sslot[i * tj + j];
            const double t = (s >= 0) ? tau[(long)s * nr + r] : 0.0;
#pragma unroll
            for (int q = 0; q < TK; ++q) acc[i][q] = fma(t, av[q], acc[i][q]);
        }
    }
#pragma unroll
    for (int i = 0; i < TI; ++i) {
        if (ib + i >= ti) continue;
        double* op = out + ((long)(i0 + ib + i) * kc + kb) * nr + r;
#pragma unroll
        for (int q = 0; q < TK; ++q) if (kb + q < kc) op[(long)q * nr] = fma(-alpha, acc[i][q], op[(long)q * nr]);
    }
}
cudaError_t launch_contract(double* out, const double* a, const double* tau, const int* slot, int i0, int ti, int j0, int tj,
                            int kc, long nr, double alpha, cudaStream_t st) {
    constexpr int TI = 4, TK = 8;
    dim3 grid((unsigned)((nr + 127) / 128), (unsigned)((ti + TI - 1) / TI), (unsigned)((kc + TK - 1) / TK));
    contract_kernel<TI, TK><<<grid, 128, sizeof(int) * TI * tj, st>>>(out, a, tau, slot, i0, ti, j0, tj, kc, nr, alpha);
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

}  // namespace tddft
