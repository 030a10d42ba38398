// Launch wrappers of the non-FFT kernels (kernels.cu, gemm.cu).  All asynchronous on the given stream.
#pragma once
#include <cuda_runtime.h>
#include "common.h"

namespace tddft {

// Where the functions of one spin block of a trial-vector block live: function f = v*kc + kk is the complex
// half-sphere vector at  base + (k0 + kk)*vec_len + block_off + v*npwh   (units: complex elements).
struct FunLayout {
    long vec_len; long block_off; long npwh; int kc; int k0;
};

// S1: sphere -> zeroed complex work grids, two functions per grid (re/im), functions f0 .. f0+2*batch-1 (< nfun)
cudaError_t launch_scatter_pack2(const cplx* X, FunLayout lay, int f0, int nfun, int batch, const int* idx_p, const int* idx_m,
                                 cplx* work, long nr, cudaStream_t st);
// S6+S7: work grids -> sphere with scale, plus (kin[g] - eig[v]) * x(g)  (Eq. 3); X = null: no D term
cudaError_t launch_gather_unpack2(const cplx* work, long nr, const int* idx_p, const int* idx_m, int f0, int nfun, int batch,
                                  double scale, const cplx* X, cplx* AX, FunLayout lay, const double* kin, const double* eig,
                                  cudaStream_t st, bool accumulate = false /* X == null only: AX += result */);
// plain sphere -> grid for one function per complex grid pair is not needed; orbitals use scatter_pack2 too.

// S2: drho[kk][r] = sum_v phi[v][r] * a[v*kc+kk][r]   (inner sum of Eq. 4)
cudaError_t launch_drho(const double* phi, const double* a, int nocc, int kc, long nr, double* drho, cudaStream_t st, bool accumulate = false);
// S3 pointwise: V_s[kk][r] = vh[kk][r] + f_s0[r]*drho0[kk][r] + f_s1[r]*drho1[kk][r]  (drho1/f_s1 may be null)
cudaError_t launch_hxc_potential(const double* vh, const double* f0, const double* drho0, const double* f1, const double* drho1,
                                 int kc, long nr, double* V, cudaStream_t st);
// S5 start value: out[f][r] = phi[v][r]*V[kk][r] (if V) + vloc[r]*a[f][r] (if vloc), f = v*kc+kk
// ftot = functions per chunk of a/out when the nocc*kc functions are the first part of a larger batch (<= 0: nocc*kc)
cudaError_t launch_out_init(const double* phi, const double* V, const double* vloc, const double* a, int nocc, int kc, long nr,
                            double* out, cudaStream_t st, long ftot = 0);
// S5 (Eq. 6) on batches in the chunked layout [nr/32][function][32] (common.h); ftot = functions in
// a/out (nocc*kc), stot = slots in the tau tile.
// Register-resident tiles (contract.cu): one launch does a whole tile with up to contract_full_max_tile() rows (any number of
// columns); contract_full_pref_tile() is the edge the default plan uses (the largest one whose kernel keeps registers free for
// running fragment loads ahead of the DMMAs).  diag: ti == tj, same orbital block, tau packed upper-triangular (one direction,
// symmetric reads); else dense slots i*tj + j and both directions.
int contract_full_max_tile();
int contract_full_pref_tile();
cudaError_t launch_contract_full(bool diag, double* out, const double* a, const double* tau, int i0, int ti, int j0, int tj, int kc,
                                 long ftot, long stot, long nr, double alpha, cudaStream_t st);
// spin-flip K1e potential V[kk][r] = f[r] * d[kk][r] (Eq. 24); D term alone AX = (kin - eig_v) X (Eq. 3)
cudaError_t launch_scale_potential(const double* f, const double* d, int kc, long nr, double* V, cudaStream_t st);
cudaError_t launch_d_term(const cplx* X, cplx* AX, FunLayout lay, int nfun, const double* kin, const double* eig, cudaStream_t st);
// out[f0 + (t - t_first)*fstep] += scale * sum_j M[j] * tau[j*nt + t], t_first <= t < t_first + t_count (Eq. 7 / Eq. 28 band sums)
cudaError_t launch_pattern_reduce(const double* M, const double* tau, int nj, int nt, int t_first, int t_count, long nr, double* out, long ftot,
                                  long f0, long fstep, double scale, cudaStream_t st);
cudaError_t launch_square(const double* phi, long n, double* sq, cudaStream_t st);
cudaError_t launch_symmetrize(double* H, int m, double scale, cudaStream_t st);   // H <- scale (H + H^T)/2
cudaError_t launch_chol_inv(double* A, double* Linv, int n, int* status, cudaStream_t st);
cudaError_t launch_sf_kernel_table(const double* rho_up, const double* rho_dn, long nr, double rho_floor, double cut, double* fsf,
                                   cudaStream_t st);
// S0: rho[r] = sum_v phi[v][r]^2 ; LDA kernel f_xc (Eq. 8; reading A5)
cudaError_t launch_rho0(const double* phi, int nocc, long nr, double* rho, cudaStream_t st);
cudaError_t launch_lda_fxc(const double* rho_up, const double* rho_dn, long nr, double rho_floor, double* fuu, double* fud,
                           double* fdd, cudaStream_t st);

// ---- dense contractions on FP64 tensor cores (gemm.cu) ------------------------------------------------
// C[m][n] (ldc) = cscale * sum_k w_k A[m][k] B[n][k], A rows at lda, B row n at  B + (n / bgrp)*bstride_grp + (n % bgrp)*ldb.
// w_k = 1/2 where k % wperiod == 0 (wperiod > 0), else 1: with cscale = 2 this is the Gamma-point inner product.
// K may be split over `splits` CTAs along k; partial sums go to `partial` [splits][m][n] and are reduced in order.
cudaError_t launch_gemm_nt(const double* A, long lda, const double* B, long ldb, int bgrp, long bstride_grp, double* C, long ldc,
                           int M, int N, long K, long wperiod, double cscale, int splits, double* partial, cudaStream_t st);
int gemm_nt_tile_count(int M, int N);   // CTAs per k split of launch_gemm_nt (for choosing splits that fill the SMs)
// S_b[u][u'] = <phi_u| (T - lam_b)^-1 |phi_u'> (Gamma inner product, |T - lam| floored at dfloor keeping sign) for nb shifts;
// Phi [M][K] with K = 2 npwh reals, kin [npwh], lam device [nb], S [nb][M][M]  (reading A11b: projector-aware Davidson correction)
cudaError_t launch_gram_shift(const double* Phi, long lda, int M, long K, const double* kin, const double* lam, int nb, double dfloor,
                              double* S, cudaStream_t st);
// C[m][n] += cscale * sum_k At[k][m] B[k][n];  C row m at  C + (m / cgrp)*cstride_grp + (m % cgrp)*ldc
cudaError_t launch_gemm_tn_acc(const double* At, long ldat, const double* B, long ldb, double* C, long ldc, int cgrp,
                               long cstride_grp, int M, long N, int K, double cscale, cudaStream_t st);

}  // namespace tddft
