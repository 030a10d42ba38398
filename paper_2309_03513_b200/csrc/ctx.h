// The context behind the C ABI and the internal driver interface shared by api.cu, extensions.cu and davidson.cu.
#pragma once
#include <string>
#include <vector>
#include "common.h"
#include "kernels.h"
#include "plan.h"

struct TileInfo {
    int i0, ti, j0, tj;        // row block [i0, i0+ti), column block [j0, j0+tj), i0 <= j0
    long pair_off; int npairs; // kept pairs (i <= j) of this tile inside PairTiles::d_pairs
    bool diag;                 // same orbital block on both sides: tau packed upper-triangular
    bool partial;              // a pair mask dropped some pairs of the tile: their tau slots must read as zero
    long nslots;               // tau slots of the tile (dense ti*tj, or ti(ti+1)/2 on the diagonal)
};
struct PairTiles {
    int T = 0, W = 0, nocc = 0;
    std::vector<TileInfo> tiles;
    std::vector<int> owner;    // shard that applies each tile (all 0 without sharding)
    int2* d_pairs = nullptr;   // pairs in processing order (sub-blocks of sbi x sbj, so a batch touches few orbitals)
    int* d_pslot = nullptr;    // tau slot of each pair of d_pairs
    int sbi = 0, sbj = 0, batch_pairs = 0;
    long max_pairs = 0, total_pairs = 0;
};

struct StageEvent { int stage; cudaEvent_t beg, end; };

struct tddft_ctx {
    tddft::HostPlan hp;
    int device = 0;
    double ecut = 0, alpha = 0;
    int nspin = 1, nocc[2] = {0, 0};
    const double* psi[2] = {nullptr, nullptr};
    std::vector<double> eig_h[2];
    // options
    int use_hartree_fxc = 1;
    double rho_floor = 1e-10;
    const double* vloc[2] = {nullptr, nullptr};
    cudaStream_t stream = nullptr;
    double workspace_gb = 0;
    double work_l2_mb = 48.0;        // launches with smaller work grids keep them under the normal L2 policy
    int pair_tile = 0, fft_batch = 0, tile_width = 0, plan = 0;
    int shard_rank = 0, shard_count = 1;   // sharding of one apply over GPUs: this context owns the tiles with owner == shard_rank
    int num_sms = 148;
    int prefer_cluster = 0;          // fft_path = 2: two-CTA cluster plane kernels where a shape has both variants
    bool fused = false;              // the grid shape has fused plane/x kernels (fft_fused.cu) and they are not switched off
    int dav_max_subspace = 0, dav_max_iter = 0, dav_block = 0, dav_precond = 0, verbose = 0;
    double dav_tol = 0; const double* dav_x0 = nullptr; int dav_nx0 = 0;
    unsigned long long seed = 0;
    int sf_xc = 0; double sf_cut = 1e-3;
    // device tables
    int *d_idx_p = nullptr, *d_idx_m = nullptr;
    int* d_cmap[2] = {nullptr, nullptr};   // fused path: pruned column maps (plan.h), kind 0 = products, 1 = sphere functions
    double *d_kin = nullptr, *d_vc = nullptr, *d_eig[2] = {nullptr, nullptr};
    tddft::cplx* d_tw[3] = {nullptr, nullptr, nullptr};
    // Real-space orbitals the grid part of the operator runs on: phi_v, or the rotated phi~_n of Eq. 31 when wannier_u is given
    // (every real-space term is covariant under the rotation).  phi_shared: both spins use ONE buffer (d_phi[0] == d_phi[1]) that
    // holds the orbitals of spin phi_spin and is refilled on demand (configurations whose orbitals do not fit twice).
    double* d_phi[2] = {nullptr, nullptr};
    bool phi_shared = false; int phi_spin = -1;
    double* d_U[2] = {nullptr, nullptr};    // [v][n] and its transpose [n][v], device; null = no rotation
    double* d_Ut[2] = {nullptr, nullptr};
    std::vector<char> mask[2];              // [nocc*nocc] kept pairs of the exchange orbitals; empty = all
    double* d_fxc[3] = {nullptr, nullptr, nullptr};
    double* d_fsf = nullptr;                // spin-flip kernel table of Eq. 26 (only with sf_xc)
    tddft::cplx* d_work = nullptr;   // [fft_batch][nr]
    // ACE (Eqs. 28-30): xi_k of each spin in the half-sphere storage, [n_ace][npwh]
    int n_ace[2] = {0, 0};
    tddft::cplx* d_xi[2] = {nullptr, nullptr};
    // per-call workspace arena
    char* arena = nullptr; size_t arena_bytes = 0;
    PairTiles tiles[2];
    // host-buffer entry point: copies run on their own stream, block by block, behind the kernels (api.cu)
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_x_ready[2] = {nullptr, nullptr}, ev_ax_done[2] = {nullptr, nullptr};
    double *host_dx = nullptr, *host_dax = nullptr; size_t host_bytes = 0;   // device staging of the host entry point (kept between calls)
    bool overlap_copies = false;     // set only while tddft_apply_liouville_host drives an apply
    // bookkeeping
    tddft_stats stats{};
    int last_pair_batch = 0, last_pair_tile = 0, last_tile_width = 0, last_kc = 0, last_resident = 1;
    bool timing = false;
    std::vector<StageEvent> events;
    std::string err;
};

namespace tddft {
int set_err(tddft_ctx* c, int status, const std::string& msg);
int apply_liouville_dev(tddft_ctx* c, const double* X, double* AX, int nvec, int mode);
long vector_len(const tddft_ctx* c, int mode);
// Yout[row] += scale * sum_u basis_u <basis_u|Yin[row]> (Gamma inner product) for functions laid out as rows: row n of Y at
// Y + (n / grp)*grp_stride + (n % grp)*2*npwh (doubles), same layout for Yin and Yout; basis [nb][npwh] complex; scratch O.
// P_c: basis = psi, Yin = Yout, scale = -1.  ACE term of D (Eq. 29): basis = xi, Yin = X, Yout = AX, scale = -alpha.
int lowrank_rows(tddft_ctx* c, const double* basis, int nb, const double* Yin, double* Yout, int nrows, int grp, long grp_stride,
                 double scale, double* O, size_t o_cap);
int project_rows(tddft_ctx* c, int tgt_spin, double* Y, int nrows, int grp, long grp_stride, double* O, size_t o_cap);
size_t project_scratch_doubles(const tddft_ctx* c, int maxocc, int nrows, size_t max_bytes);   // capacity (doubles) project_rows wants for O
int ensure_arena(tddft_ctx* c, size_t bytes);
int ensure_phi(tddft_ctx* c, int spin);      // makes d_phi[spin] hold that spin's orbitals (phi_shared mode refills)
size_t workspace_budget(const tddft_ctx* c);
// real space <-> sphere on batches of functions (api.cu)
int to_real_space(tddft_ctx* c, const cplx* X, FunLayout lay, int nfun, double* dst, int chunked, long fbase0 = 0, long ftotal = 0);
int to_sphere_plus_d(tddft_ctx* c, const double* src, int nfun, const cplx* X, cplx* AX, FunLayout lay, const double* d_eig, long fbase0 = 0,
                     long ftotal = 0, bool accumulate = false);
int hartree(tddft_ctx* c, const double* d0, const double* d1, double scale, int kc, double* vh);
// tau_p = C[A1[x_p] A2[y_p]] for npairs pairs (device lists), written to slot d_slots[p] (or p) of a batch of stot functions
int pair_potentials_dev(tddft_ctx* c, const double* A1, const double* A2, const int2* d_pairs, const int* d_slots, long npairs,
                        int batch_pairs, double* tau, int chunked, long stot);
int build_tiles(tddft_ctx* c, int spin, int T, int W);
int orbital_overlap(tddft_ctx* c, int spin, double* S);     // Eq. 32, HOST S [N][N]
// extensions.cu: ACE construction (Eqs. 28-30) from the occupied orbitals plus n_extra further ones (device [n_extra][npwh])
int build_ace(tddft_ctx* c, int spin, const double* psi_extra, int n_extra);
// stage timing (api.cu)
enum { ST_S1 = 0, ST_S23, ST_S4, ST_S5, ST_S6, ST_S8, ST_S7X, ST_COUNT };
struct StageTimer {
    tddft_ctx* c; int idx = -1;
    StageTimer(tddft_ctx* c_, int stage);
    ~StageTimer();
};
void collect_timing(tddft_ctx* c);
}  // namespace tddft

#define TD_CUDA(c, call)                                                                                   \
    do {                                                                                                   \
        cudaError_t e_ = (call);                                                                           \
        if (e_ != cudaSuccess)                                                                             \
            return tddft::set_err((c), TDDFT_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));   \
    } while (0)
#define TD_RC(call) do { int rc_ = (call); if (rc_) return rc_; } while (0)
