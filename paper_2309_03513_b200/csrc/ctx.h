// The context behind the C ABI and the internal driver interface shared by api.cu and davidson.cu.
#pragma once
#include <string>
#include <vector>
#include "common.h"
#include "kernels.h"
#include "plan.h"

struct TileInfo {
    int i0, ti, j0, tj;        // row block [i0, i0+ti), column block [j0, j0+tj), i0 <= j0
    long pair_off; int npairs; // unique pairs (i <= j) of this tile inside PairTiles::d_pairs
    long slot_off, slotT_off;  // slot tables [ti][tj] and (off-diagonal tiles) [tj][ti] inside d_slot
};
struct PairTiles {
    int T = 0, nocc = 0;
    std::vector<TileInfo> tiles;
    int2* d_pairs = nullptr;   // pairs in processing order (sub-blocks of sbi x sbj, so a batch touches few orbitals)
    int* d_pslot = nullptr;    // tau slot of each pair of d_pairs
    int* d_slot = nullptr;
    int sbi = 0, sbj = 0, batch_pairs = 0;
    long max_pairs = 0;
};

struct StageEvent { int stage; cudaEvent_t beg, end; };

struct tddft_ctx {
    tddft::HostPlan hp;
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
    int pair_tile = 0, fft_batch = 0;
    int num_sms = 148;
    bool ct_full = true;             // S5 with the register-resident tile kernel (kernels.cu); TDDFT_CT_FULL=0 selects the row-block kernels
    bool fused = false;              // the grid shape has fused plane/x kernels (fft_fused.cu) and they are not switched off
    int dav_max_subspace = 0, dav_max_iter = 0; double dav_tol = 0; const double* dav_x0 = nullptr; int dav_nx0 = 0;
    unsigned long long seed = 0;
    // device tables
    int *d_idx_p = nullptr, *d_idx_m = nullptr;
    int* d_cmap[2] = {nullptr, nullptr};   // fused path: pruned column maps (plan.h), kind 0 = products, 1 = sphere functions
    double *d_kin = nullptr, *d_vc = nullptr, *d_eig[2] = {nullptr, nullptr};
    tddft::cplx* d_tw[3] = {nullptr, nullptr, nullptr};
    double* d_phi[2] = {nullptr, nullptr};
    double* d_fxc[3] = {nullptr, nullptr, nullptr};
    tddft::cplx* d_work = nullptr;   // [fft_batch][nr]
    double* d_zeros = nullptr;       // 1 KB of zeros (source of padding rows for the contraction's bulk copies)
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
    int last_pair_batch = 0, last_pair_tile = 0;
    bool timing = false;
    std::vector<StageEvent> events;
    std::string err;
};

namespace tddft {
int set_err(tddft_ctx* c, int status, const std::string& msg);
int apply_liouville_dev(tddft_ctx* c, const double* X, double* AX, int nvec, int mode);
long vector_len(const tddft_ctx* c, int mode);
// P_c on functions laid out as rows: row n at Y + (n / grp)*grp_stride + (n % grp)*2*npwh (doubles); scratch O from arena
int project_rows(tddft_ctx* c, int tgt_spin, double* Y, int nrows, int grp, long grp_stride, double* O, size_t o_cap);
size_t project_scratch_doubles(const tddft_ctx* c, int maxocc, int nrows, size_t max_bytes);   // capacity (doubles) project_rows wants for O
int ensure_arena(tddft_ctx* c, size_t bytes);
}  // namespace tddft

#define TD_CUDA(c, call)                                                                                   \
    do {                                                                                                   \
        cudaError_t e_ = (call);                                                                           \
        if (e_ != cudaSuccess)                                                                             \
            return tddft::set_err((c), TDDFT_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));   \
    } while (0)
