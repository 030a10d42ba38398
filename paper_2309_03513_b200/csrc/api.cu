// C ABI of the library and the driver of one Liouville application.
// Product path: every numerical step below is a kernel launch; the host only orchestrates.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include "ctx.h"

using namespace tddft;

static std::string g_init_error;

namespace tddft {

int set_err(tddft_ctx* c, int status, const std::string& msg) {
    if (c) c->err = msg; else g_init_error = msg;
    return status;
}

long vector_len(const tddft_ctx* c, int mode) {
    if (mode == TDDFT_SPIN_CONSERVING) {
        long n = 0;
        for (int s = 0; s < c->nspin; ++s) n += (long)c->nocc[s] * c->hp.npwh;
        return n;
    }
    if (c->nspin != 2) return -1;
    return (long)c->nocc[mode == TDDFT_SPIN_FLIP ? 0 : 1] * c->hp.npwh;
}

int ensure_arena(tddft_ctx* c, size_t bytes) {
    if (bytes <= c->arena_bytes) return TDDFT_OK;
    if (c->arena) { cudaFree(c->arena); c->arena = nullptr; c->arena_bytes = 0; }
    cudaError_t e = cudaMalloc((void**)&c->arena, bytes);
    if (e != cudaSuccess) { cudaGetLastError(); return set_err(c, TDDFT_ENOMEM, "device workspace allocation failed"); }
    c->arena_bytes = bytes;
    return TDDFT_OK;
}

// ---- stage timing ---------------------------------------------------------------------------------
enum { ST_S1 = 0, ST_S23, ST_S4, ST_S5, ST_S6, ST_S8, ST_COUNT };
struct StageTimer {
    tddft_ctx* c; int idx = -1;
    StageTimer(tddft_ctx* c_, int stage) : c(c_) {
        if (!c->timing) return;
        StageEvent ev; ev.stage = stage;
        cudaEventCreate(&ev.beg); cudaEventCreate(&ev.end);
        cudaEventRecord(ev.beg, c->stream);
        c->events.push_back(ev); idx = (int)c->events.size() - 1;
    }
    ~StageTimer() { if (idx >= 0) cudaEventRecord(c->events[idx].end, c->stream); }
};
static void collect_timing(tddft_ctx* c) {
    if (!c->timing) return;
    cudaStreamSynchronize(c->stream);
    double ms[ST_COUNT] = {0};
    for (auto& ev : c->events) {
        float t = 0; cudaEventElapsedTime(&t, ev.beg, ev.end);
        ms[ev.stage] += t;
        cudaEventDestroy(ev.beg); cudaEventDestroy(ev.end);
    }
    c->events.clear();
    c->stats.ms_s1_to_real = ms[ST_S1]; c->stats.ms_s23_hxc = ms[ST_S23]; c->stats.ms_s4_pair_fft = ms[ST_S4];
    c->stats.ms_s5_contract = ms[ST_S5]; c->stats.ms_s6_to_sphere = ms[ST_S6]; c->stats.ms_s8_project = ms[ST_S8];
    c->stats.ms_total = 0; for (int i = 0; i < ST_COUNT; ++i) c->stats.ms_total += ms[i];
}

// ---- FFT pass sequences ---------------------------------------------------------------------------
static SArgs ypass_args(const tddft_ctx* c, int batch) {
    const int* n = c->hp.n;
    SArgs a{}; a.n = n[1]; a.stride = n[2]; a.inner = n[2]; a.nouter = n[0]; a.outer_stride = (long)n[1] * n[2];
    a.nr = c->hp.nr; a.batch = batch; a.tw = c->d_tw[1]; a.work = c->d_work; a.ktab = nullptr;
    return a;
}
// Frequency-space work grids: full scrambled grids on the general path; on the fused path only the live (ky,kz)
// columns of the transform's kind (plan.h: KIND_PROD = products of two sphere functions, KIND_SPHERE = sphere functions).
enum { KIND_PROD = 0, KIND_SPHERE = 1 };
static long work_stride(const tddft_ctx* c, int kind) { return c->fused ? (long)c->hp.n[0] * c->hp.ncols[kind] : c->hp.nr; }
static SArgs xpass_args(const tddft_ctx* c, int batch, int kind) {
    const int* n = c->hp.n;
    const long inner = c->fused ? c->hp.ncols[kind] : (long)n[1] * n[2];
    SArgs a{}; a.n = n[0]; a.stride = inner; a.inner = inner; a.nouter = 1; a.outer_stride = 0;
    a.nr = work_stride(c, kind); a.batch = batch; a.tw = c->d_tw[0]; a.work = c->d_work; a.ktab = c->d_vc;
    return a;
}
static ZArgs zpass_args(const tddft_ctx* c, int batch, int kind) {
    const int* n = c->hp.n;
    ZArgs a{}; a.n = n[2]; a.npencils = (long)n[0] * n[1]; a.nr = c->hp.nr; a.batch = batch; a.tw = c->d_tw[2]; a.tw2 = c->d_tw[1]; a.work = c->d_work;
    a.lscale = 1.0; a.sscale = 1.0;
    a.cmap = c->d_cmap[kind]; a.ncols = c->hp.ncols[kind]; a.wstride = work_stride(c, kind);
    return a;
}

// The three legs of every transform: (y,z) forward with a fused load, the x pass (forward / inverse / forward *
// Coulomb table * inverse), (y,z) inverse with a fused split store.  Fused plane/x kernels when the grid shape has
// them (fft_fused.cu), otherwise one general pass kernel per axis.
static int leg_forward_yz(tddft_ctx* c, int lkind, const ZArgs& z) {
    if (c->fused) { TD_CUDA(c, launch_plane(c->hp.n[1], c->hp.n[2], false, lkind, ZS_WORK, z, c->stream)); c->stats.kernel_launches += 1; return TDDFT_OK; }
    TD_CUDA(c, launch_zpass(false, lkind, ZS_WORK, z, c->stream));
    TD_CUDA(c, launch_spass(SM_FWD, ypass_args(c, z.batch), c->stream));
    c->stats.kernel_launches += 2;
    return TDDFT_OK;
}
static int leg_x(tddft_ctx* c, int mode, int nb, int kind) {
    if (c->fused) TD_CUDA(c, launch_xpass(mode, xpass_args(c, nb, kind), c->stream));
    else TD_CUDA(c, launch_spass(mode, xpass_args(c, nb, kind), c->stream));
    c->stats.kernel_launches += 1;
    return TDDFT_OK;
}
static int leg_inverse_yz(tddft_ctx* c, const ZArgs& z) {
    if (c->fused) { TD_CUDA(c, launch_plane(c->hp.n[1], c->hp.n[2], true, ZL_WORK, ZS_SPLIT2, z, c->stream)); c->stats.kernel_launches += 1; return TDDFT_OK; }
    TD_CUDA(c, launch_spass(SM_INV, ypass_args(c, z.batch), c->stream));
    TD_CUDA(c, launch_zpass(true, ZL_WORK, ZS_SPLIT2, z, c->stream));
    c->stats.kernel_launches += 2;
    return TDDFT_OK;
}
#define TD_RC(call) do { int rc_ = (call); if (rc_) return rc_; } while (0)

// tau_p = C[phi_i phi_j] for npairs pairs (device list), two pairs per complex grid
// d_slots (optional): tau slot of each pair; null = slot p for pair p.  batch_pairs <= 2*fft_batch pairs per launch.
static int pair_potentials_dev(tddft_ctx* c, const double* phi, const int2* d_pairs, const int* d_slots, long npairs, int batch_pairs, double* tau, int chunked) {
    const long nr = c->hp.nr;
    for (long p0 = 0; p0 < npairs; p0 += batch_pairs) {
        const int np = (int)std::min<long>(batch_pairs, npairs - p0);
        const int nb = (np + 1) / 2;
        ZArgs z = zpass_args(c, nb, KIND_PROD);
        z.phi = phi; z.pairs = d_pairs + p0; z.npairs = np;
        TD_RC(leg_forward_yz(c, ZL_PAIR, z));
        TD_RC(leg_x(c, SM_CONV, nb, KIND_PROD));
        z.dst = tau; z.nfun = np; z.sscale = 1.0; z.chunked = chunked; z.fbase = d_slots ? 0 : p0; z.ftotal = npairs;
        z.slots = d_slots ? d_slots + p0 : nullptr;
        TD_RC(leg_inverse_yz(c, z));
        c->stats.pair_ffts += np;
    }
    return TDDFT_OK;
}

// S1: nfun half-sphere functions -> real space, dst[f][r] = Omega^-1/2 sum_G c_f(G) exp(i G.r)
static int to_real_space(tddft_ctx* c, const cplx* X, FunLayout lay, int nfun, double* dst, int chunked) {
    const long nr = c->hp.nr;
    const double scale = 1.0 / std::sqrt(c->hp.omega);
    for (int f0 = 0; f0 < nfun; f0 += 2 * c->fft_batch) {
        const int nf = std::min(2 * c->fft_batch, nfun - f0);
        const int nb = (nf + 1) / 2;
        TD_CUDA(c, launch_scatter_pack2(X, lay, f0, nfun, nb, c->d_idx_p, c->d_idx_m, c->d_work, work_stride(c, KIND_SPHERE), c->stream));
        TD_RC(leg_x(c, SM_INV, nb, KIND_SPHERE));
        ZArgs z = zpass_args(c, nb, KIND_SPHERE);
        z.dst = dst; z.nfun = nf; z.sscale = scale; z.chunked = chunked; z.fbase = f0; z.ftotal = nfun;
        TD_RC(leg_inverse_yz(c, z));
        c->stats.kernel_launches += 1;
    }
    return TDDFT_OK;
}

// S6+S7: real-space functions -> half sphere, AX = (Omega^1/2/N_r) FFT[src] + (|G|^2/2 - eps_v) X
static int to_sphere_plus_d(tddft_ctx* c, const double* src, int nfun, const cplx* X, cplx* AX, FunLayout lay, const double* d_eig) {
    const long nr = c->hp.nr;
    const double scale = std::sqrt(c->hp.omega) / (double)nr;
    for (int f0 = 0; f0 < nfun; f0 += 2 * c->fft_batch) {
        const int nf = std::min(2 * c->fft_batch, nfun - f0);
        const int nb = (nf + 1) / 2;
        ZArgs z = zpass_args(c, nb, KIND_SPHERE);
        z.src0 = src; z.src1 = nullptr; z.nfun = nf; z.lscale = 1.0; z.chunked = 1; z.fbase = f0; z.ftotal = nfun;
        TD_RC(leg_forward_yz(c, ZL_PACK2, z));
        TD_RC(leg_x(c, SM_FWD, nb, KIND_SPHERE));
        TD_CUDA(c, launch_gather_unpack2(c->d_work, work_stride(c, KIND_SPHERE), c->d_idx_p, c->d_idx_m, f0, nfun, nb, scale, X, AX, lay, c->d_kin, d_eig, c->stream));
        c->stats.kernel_launches += 1;
    }
    return TDDFT_OK;
}

// S3 Hartree part: vh[kk] = C[scale * (d0[kk] + d1[kk])]
static int hartree(tddft_ctx* c, const double* d0, const double* d1, double scale, int kc, double* vh) {
    const long nr = c->hp.nr;
    for (int f0 = 0; f0 < kc; f0 += 2 * c->fft_batch) {
        const int nf = std::min(2 * c->fft_batch, kc - f0);
        const int nb = (nf + 1) / 2;
        ZArgs z = zpass_args(c, nb, KIND_PROD);
        z.src0 = d0; z.src1 = d1; z.nfun = nf; z.lscale = scale; z.chunked = 0; z.fbase = f0; z.ftotal = kc;
        TD_RC(leg_forward_yz(c, ZL_PACK2, z));
        TD_RC(leg_x(c, SM_CONV, nb, KIND_PROD));
        z.dst = vh; z.sscale = 1.0;
        TD_RC(leg_inverse_yz(c, z));
    }
    return TDDFT_OK;
}

// S8: rows <- P_c rows with the occupied orbitals of tgt_spin, two tensor-core GEMMs
int project_rows(tddft_ctx* c, int tgt, double* Y, int nrows, int grp, long grp_stride, double* O, size_t o_cap) {
    const long k2 = 2 * c->hp.npwh;
    const int no = c->nocc[tgt];
    const long ldo = (nrows + 1) & ~1L;                      // even pitch: 16-byte aligned rows for the async copies
    // k splits chosen so that the CTAs fill whole waves of the SMs (ordered reduction, deterministic)
    const long tiles = gemm_nt_tile_count(no, nrows);
    int splits = 1; double best = 0.0;
    for (int s = 1; s <= 16; ++s) {
        if ((size_t)no * ldo + (size_t)s * no * nrows > o_cap || k2 / s < 256) break;
        const long ctas = tiles * s, waves = (ctas + c->num_sms - 1) / c->num_sms;
        const double eff = (double)ctas / (double)(waves * c->num_sms);
        if (eff > best + 0.02) { best = eff; splits = s; }
    }
    double* partial = splits > 1 ? O + (size_t)no * ldo : nullptr;
    TD_CUDA(c, launch_gemm_nt(c->psi[tgt], k2, Y, k2, grp, grp_stride, O, ldo, no, nrows, k2, k2, 2.0, splits, partial, c->stream));
    TD_CUDA(c, launch_gemm_tn_acc(O, ldo, c->psi[tgt], k2, Y, k2, grp, grp_stride, nrows, k2, no, -1.0, c->stream));
    c->stats.kernel_launches += 2 + (splits > 1 ? 1 : 0);
    return TDDFT_OK;
}
size_t project_scratch_doubles(const tddft_ctx* c, int maxocc, int nrows, size_t max_bytes) {
    const size_t one = (size_t)maxocc * ((nrows + 1) & ~1L);
    size_t cap = std::min<size_t>((size_t)1 << 28, max_bytes / 8 / sizeof(double));   // k-split partial sums: <= 2 GB and <= 1/8 of the budget
    int mult = 13;
    while (mult > 1 && one * mult > cap) --mult;
    return one * mult;
}

// ---- pair tiles -------------------------------------------------------------------------------------
// sub-block of si rows x sj columns (sj even, si*sj <= cap pairs): few orbital grids per pair, launch well filled
static void choose_subblock(int cap, int* si_out, int* sj_out) {
    double best = 1e300;
    *si_out = 1; *sj_out = std::max(2, cap & ~1);
    for (int sj = 2; sj <= cap; sj += 2)
        for (int si = 1; si * sj <= cap; ++si) {
            const double fill = (double)(si * sj) / cap;
            const double cost = (double)(si + sj) / (si * sj) / (fill * fill);
            if (cost < best) { best = cost; *si_out = si; *sj_out = sj; }
        }
}
static int build_tiles(tddft_ctx* c, int spin, int T) {
    PairTiles& pt = c->tiles[spin];
    const int N = c->nocc[spin];
    if (pt.T == T && pt.nocc == N && pt.d_pairs) return TDDFT_OK;
    if (pt.d_pairs) cudaFree(pt.d_pairs);
    if (pt.d_slot) cudaFree(pt.d_slot);
    if (pt.d_pslot) cudaFree(pt.d_pslot);
    pt = PairTiles{};
    pt.T = T; pt.nocc = N;
    // Processing order: sub-blocks of sbi rows x sbj columns (sbj even, sbi*sbj <= one launch of 2*fft_batch pairs), row-major
    // inside a sub-block.  A launch then multiplies sbi + sbj orbital grids (L2 resident) instead of ~2*fft_batch, and the two
    // pairs packed into one complex grid still share their first orbital.
    choose_subblock(2 * c->fft_batch, &pt.sbi, &pt.sbj);
    pt.batch_pairs = pt.sbi * pt.sbj;
    const int nb = (N + T - 1) / T;
    std::vector<int2> pairs; std::vector<int> slot, pslot;
    for (int bi = 0; bi < nb; ++bi)
        for (int bj = bi; bj < nb; ++bj) {
            TileInfo t{};
            t.i0 = bi * T; t.ti = std::min(T, N - t.i0); t.j0 = bj * T; t.tj = std::min(T, N - t.j0);
            t.pair_off = (long)pairs.size(); t.slot_off = (long)slot.size();
            std::vector<int> s((size_t)t.ti * t.tj, -1);
            int cnt = 0;
            for (int i = 0; i < t.ti; ++i)
                for (int j = 0; j < t.tj; ++j) {
                    const int gi = t.i0 + i, gj = t.j0 + j;
                    if (gi > gj) continue;
                    s[(size_t)i * t.tj + j] = cnt++;     // tau slots stay row-major (the contraction's layout)
                }
            for (int si0 = 0; si0 < t.ti; si0 += pt.sbi)
                for (int sj0 = 0; sj0 < t.tj; sj0 += pt.sbj)
                    for (int i = si0; i < std::min(si0 + pt.sbi, t.ti); ++i)
                        for (int j = sj0; j < std::min(sj0 + pt.sbj, t.tj); ++j) {
                            const int gi = t.i0 + i, gj = t.j0 + j;
                            if (gi > gj) continue;
                            pairs.push_back(make_int2(gi, gj));
                            pslot.push_back(s[(size_t)i * t.tj + j]);
                        }
            if (bi == bj) for (int i = 0; i < t.ti; ++i) for (int j = 0; j < i; ++j) s[(size_t)i * t.tj + j] = s[(size_t)j * t.tj + i];
            t.npairs = cnt;
            slot.insert(slot.end(), s.begin(), s.end());
            t.slotT_off = -1;
            if (bi != bj) {
                t.slotT_off = (long)slot.size();
                for (int j = 0; j < t.tj; ++j) for (int i = 0; i < t.ti; ++i) slot.push_back(s[(size_t)i * t.tj + j]);
            }
            pt.max_pairs = std::max<long>(pt.max_pairs, cnt);
            pt.tiles.push_back(t);
        }
    TD_CUDA(c, cudaMalloc((void**)&pt.d_pairs, sizeof(int2) * pairs.size()));
    TD_CUDA(c, cudaMalloc((void**)&pt.d_slot, sizeof(int) * slot.size()));
    TD_CUDA(c, cudaMalloc((void**)&pt.d_pslot, sizeof(int) * pslot.size()));
    TD_CUDA(c, cudaMemcpyAsync(pt.d_pslot, pslot.data(), sizeof(int) * pslot.size(), cudaMemcpyHostToDevice, c->stream));
    TD_CUDA(c, cudaMemcpyAsync(pt.d_pairs, pairs.data(), sizeof(int2) * pairs.size(), cudaMemcpyHostToDevice, c->stream));
    TD_CUDA(c, cudaMemcpyAsync(pt.d_slot, slot.data(), sizeof(int) * slot.size(), cudaMemcpyHostToDevice, c->stream));
    TD_CUDA(c, cudaStreamSynchronize(c->stream));   // host vectors go out of scope
    return TDDFT_OK;
}

// ---- one application ------------------------------------------------------------------------------
struct Block { int src, tgt; long off; };   // occupied spin, target spin, offset (complex) inside a trial vector

int apply_liouville_dev(tddft_ctx* c, const double* Xd, double* AXd, int nvec, int mode) {
    if (!c) return TDDFT_EINVAL;
    if (!Xd || !AXd || nvec < 1) return set_err(c, TDDFT_EINVAL, "apply: null buffer or nvec < 1");
    if (Xd == AXd) return set_err(c, TDDFT_EINVAL, "apply: AX must not alias X");
    if (mode < 0 || mode > 2) return set_err(c, TDDFT_EINVAL, "apply: unknown mode");
    if (mode != TDDFT_SPIN_CONSERVING && c->nspin != 2) return set_err(c, TDDFT_EINVAL, "spin flip needs nspin = 2");
    const cplx* X = (const cplx*)Xd; cplx* AX = (cplx*)AXd;
    const long nr = c->hp.nr, npwh = c->hp.npwh, L = vector_len(c, mode);
    c->stats = tddft_stats{};
    std::vector<Block> blocks;
    if (mode == TDDFT_SPIN_CONSERVING) { long off = 0; for (int s = 0; s < c->nspin; ++s) { blocks.push_back({s, s, off}); off += (long)c->nocc[s] * npwh; } }
    else { const int src = (mode == TDDFT_SPIN_FLIP) ? 0 : 1; blocks.push_back({src, 1 - src, 0}); }
    const bool hxc = (mode == TDDFT_SPIN_CONSERVING) && c->use_hartree_fxc;
    int maxocc = 0, sumocc = 0;
    for (auto& b : blocks) { maxocc = std::max(maxocc, std::max(c->nocc[b.src], c->nocc[b.tgt])); sumocc += c->nocc[b.src]; }

    // ---- workspace plan: k chunk kc and tile edge T under the budget --------------------------------
    size_t budget;
    {
        size_t fr = 0, tot = 0; cudaMemGetInfo(&fr, &tot);
        budget = (size_t)(0.85 * (double)(fr + c->arena_bytes));
        if (c->workspace_gb > 0) budget = std::min(budget, (size_t)(c->workspace_gb * 1073741824.0));
    }
    int kc = nvec, T = 0;
    size_t fixed = 0;
    const size_t grid_b = sizeof(double) * (size_t)chunked_elems(1, nr);   // one real grid, padded to whole chunks
    for (;;) {
        fixed = grid_b * (size_t)kc * ((size_t)sumocc + (size_t)maxocc + (hxc ? 2 * blocks.size() + 1 : 0))
              + sizeof(double) * project_scratch_doubles(c, maxocc, kc * maxocc, budget) + 4096;
        const int tcap = c->ct_full ? contract_full_max_tile() : 128;
        T = std::min(std::min(maxocc, tcap), c->pair_tile > 0 ? std::min(c->pair_tile, tcap) : tcap);
        const int tmin = std::min(maxocc, 16);
        while (T > tmin && fixed + grid_b * (size_t)T * T > budget) T = std::max(tmin, T - 8);
        if (fixed + grid_b * (size_t)T * T <= budget) break;
        if (kc == 1) return set_err(c, TDDFT_ENOMEM, "workspace budget too small for a single trial vector");
        kc = (kc + 1) / 2;
    }
    if (c->ct_full) { const int nbk = (maxocc + T - 1) / T; T = (maxocc + nbk - 1) / nbk; }   // equal blocks: the kernel's cost follows the largest
    else if (T >= 32) T &= ~31;   // the row-block contraction gives each warp 32 rows of a tile
    int rc = ensure_arena(c, fixed + grid_b * (size_t)T * T);
    if (rc) return rc;
    char* p = c->arena;
    auto carve = [&](size_t bytes) { char* q = p; p += (bytes + 255) / 256 * 256; return (double*)q; };
    std::vector<double*> a(blocks.size());
    for (size_t b = 0; b < blocks.size(); ++b) a[b] = carve(grid_b * (size_t)kc * c->nocc[blocks[b].src]);
    double* out = carve(grid_b * (size_t)kc * maxocc);
    std::vector<double*> drho(blocks.size(), nullptr), V(blocks.size(), nullptr);
    double* vh = nullptr;
    if (hxc) { for (size_t b = 0; b < blocks.size(); ++b) { drho[b] = carve(grid_b * kc); V[b] = carve(grid_b * kc); } vh = carve(grid_b * kc); }
    const size_t o_cap = project_scratch_doubles(c, maxocc, kc * maxocc, budget);
    double* O = carve(sizeof(double) * o_cap);
    double* tau = carve(grid_b * (size_t)T * T);
    for (auto& b : blocks) { rc = build_tiles(c, b.src, std::min(T, c->nocc[b.src])); if (rc) return rc; }
    c->last_pair_tile = T; c->last_pair_batch = c->tiles[blocks[0].src].batch_pairs;

    for (int k0 = 0; k0 < nvec; k0 += kc) {
        const int kcc = std::min(kc, nvec - k0);
        // S1 (+S2): trial functions to real space, response densities
        for (size_t b = 0; b < blocks.size(); ++b) {
            const int no = c->nocc[blocks[b].src];
            FunLayout lay{L, blocks[b].off, npwh, kcc, k0};
            if (c->overlap_copies) TD_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_x_ready[b], 0));     // this block of X has arrived
            { StageTimer t(c, ST_S1); rc = to_real_space(c, X, lay, no * kcc, a[b], 1); if (rc) return rc; }
            if (hxc) { StageTimer t(c, ST_S23); TD_CUDA(c, launch_drho(c->d_phi[blocks[b].src], a[b], no, kcc, nr, drho[b], c->stream)); c->stats.kernel_launches += (kcc + 3) / 4; }
        }
        // S3: Hartree + f_xc potential (Eq. 4 with f_Hxc = v_c + f_xc)
        if (hxc) {
            StageTimer t(c, ST_S23);
            if (c->nspin == 2) {
                rc = hartree(c, drho[0], drho[1], 1.0, kcc, vh); if (rc) return rc;
                TD_CUDA(c, launch_hxc_potential(vh, c->d_fxc[0], drho[0], c->d_fxc[1], drho[1], kcc, nr, V[0], c->stream));
                TD_CUDA(c, launch_hxc_potential(vh, c->d_fxc[1], drho[0], c->d_fxc[2], drho[1], kcc, nr, V[1], c->stream));
                c->stats.kernel_launches += 2;
            } else {   // closed shell, singlet channel (reading A6): V = C[2 drho] + (f_uu + f_ud) drho
                rc = hartree(c, drho[0], nullptr, 2.0, kcc, vh); if (rc) return rc;
                TD_CUDA(c, launch_hxc_potential(vh, c->d_fxc[0], drho[0], c->d_fxc[1], drho[0], kcc, nr, V[0], c->stream));
                c->stats.kernel_launches += 1;
            }
        }
        for (size_t b = 0; b < blocks.size(); ++b) {
            const Block& bl = blocks[b];
            const int no = c->nocc[bl.src];
            const double* phi = c->d_phi[bl.src];
            { StageTimer t(c, ST_S5);
              TD_CUDA(c, launch_out_init(phi, hxc ? V[b] : nullptr, c->vloc[bl.tgt], a[b], no, kcc, nr, out, c->stream)); c->stats.kernel_launches += 1; }
            // S4 + S5: exact-exchange response, tile by tile (Eq. 6; tau_vv' of PAPER.md:230)
            if (c->alpha != 0.0) {
                const PairTiles& pt = c->tiles[bl.src];
                for (const TileInfo& t : pt.tiles) {
                    { StageTimer tm(c, ST_S4); rc = pair_potentials_dev(c, phi, pt.d_pairs + t.pair_off, pt.d_pslot + t.pair_off, t.npairs, pt.batch_pairs, tau, 1); if (rc) return rc; }
                    StageTimer tm(c, ST_S5);
                    if (c->ct_full) TD_CUDA(c, launch_contract_full(t.slotT_off < 0, out, a[b], tau, t.i0, t.ti, t.j0, t.tj, kcc, (long)no * kcc,
                                                                   t.slotT_off < 0 ? (long)t.npairs : (long)t.ti * t.tj, nr, c->alpha, c->stream));
                    else if (t.slotT_off >= 0) TD_CUDA(c, launch_contract_dual(out, a[b], tau, c->d_zeros, t.i0, t.ti, t.j0, t.tj, kcc, (long)no * kcc, nr, c->alpha, c->stream));
                    else TD_CUDA(c, launch_contract_single(out, a[b], tau, pt.d_slot + t.slot_off, c->d_zeros, t.i0, t.ti, t.j0, t.tj, kcc, (long)no * kcc, t.npairs, nr, c->alpha, c->stream));
                    c->stats.kernel_launches += (kcc + 15) / 16;
                }
            }
            // S6 + S7: back to the sphere, add D (Eq. 3 with the model H of reading A4)
            FunLayout lay{L, bl.off, npwh, kcc, k0};
            { StageTimer t(c, ST_S6); rc = to_sphere_plus_d(c, out, no * kcc, X, AX, lay, c->d_eig[bl.src]); if (rc) return rc; }
            // S8: conduction-band projector of the target spin
            { StageTimer t(c, ST_S8);
              rc = project_rows(c, bl.tgt, (double*)(AX + (long)k0 * L + bl.off), kcc * no, no, 2 * L, O, o_cap); if (rc) return rc; }
            if (c->overlap_copies) TD_CUDA(c, cudaEventRecord(c->ev_ax_done[b], c->stream));               // this block of AX is final
        }
    }
    collect_timing(c);
    return TDDFT_OK;
}

}  // namespace tddft

// =====================================================================================================
extern "C" {
#pragma GCC visibility push(default)

int tddft_enumerate_gvectors(const double* lattice, double ecut, long capacity, int* miller, double* g2, long* npwh) {
    if (!lattice || !npwh || !(ecut > 0)) return TDDFT_EINVAL;
    try {
        std::vector<int> m; std::vector<double> q;
        const long n = enumerate_half_sphere(lattice, ecut, &m, &q);
        *npwh = n;
        if ((miller || g2) && capacity < n) return TDDFT_EINVAL;
        if (miller) std::memcpy(miller, m.data(), sizeof(int) * 3 * n);
        if (g2) std::memcpy(g2, q.data(), sizeof(double) * n);
    } catch (const std::bad_alloc&) { return TDDFT_ENOMEM; }
    return TDDFT_OK;
}

int tddft_destroy(tddft_ctx* c) {
    if (!c) return TDDFT_OK;
    cudaFree(c->d_idx_p); cudaFree(c->d_idx_m); cudaFree(c->d_kin); cudaFree(c->d_vc); cudaFree(c->d_cmap[0]); cudaFree(c->d_cmap[1]);
    for (int s = 0; s < 2; ++s) { cudaFree(c->d_eig[s]); cudaFree(c->d_phi[s]); }
    for (int a = 0; a < 3; ++a) { cudaFree(c->d_tw[a]); cudaFree(c->d_fxc[a]); }
    cudaFree(c->d_work); cudaFree(c->arena); cudaFree(c->d_zeros);
    cudaFree(c->host_dx); cudaFree(c->host_dax);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    for (int i = 0; i < 2; ++i) { if (c->ev_x_ready[i]) cudaEventDestroy(c->ev_x_ready[i]); if (c->ev_ax_done[i]) cudaEventDestroy(c->ev_ax_done[i]); }
    for (int s = 0; s < 2; ++s) { cudaFree(c->tiles[s].d_pairs); cudaFree(c->tiles[s].d_slot); cudaFree(c->tiles[s].d_pslot); }
    cudaGetLastError();
    delete c;
    return TDDFT_OK;
}

int tddft_init(tddft_ctx** out, const double* lattice, const int* grid, double ecut, int nspin, const int* nocc,
               const double* psi_up, const double* psi_dn, const double* eig_up, const double* eig_dn, double alpha,
               const tddft_options* opt) {
    if (!out) return TDDFT_EINVAL;
    *out = nullptr;
    if (!lattice || !grid || !nocc || !psi_up || !eig_up) return set_err(nullptr, TDDFT_EINVAL, "init: null argument");
    if (nspin != 1 && nspin != 2) return set_err(nullptr, TDDFT_EINVAL, "init: nspin must be 1 or 2");
    if (nspin == 2 && (!psi_dn || !eig_dn)) return set_err(nullptr, TDDFT_EINVAL, "init: nspin = 2 needs psi_dn and eig_dn");
    if (!(ecut > 0) || !(alpha >= 0)) return set_err(nullptr, TDDFT_EINVAL, "init: ecut must be > 0 and alpha >= 0");
    for (int s = 0; s < nspin; ++s) if (nocc[s] < 1) return set_err(nullptr, TDDFT_EINVAL, "init: nocc must be >= 1");
    for (int a = 0; a < 3; ++a) if (grid[a] < 1) return set_err(nullptr, TDDFT_EINVAL, "init: bad grid");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return set_err(nullptr, TDDFT_ECUDA, "init: no CUDA device (this library has no CPU path)"); }
    tddft_ctx* c = nullptr;
    try { c = new tddft_ctx(); } catch (const std::bad_alloc&) { return TDDFT_ENOMEM; }
    auto fail = [&](int st, const std::string& msg) { g_init_error = msg; tddft_destroy(c); return st; };
    try {
        for (int a = 0; a < 3; ++a) if (!fft_size_supported(grid[a])) return fail(TDDFT_EUNSUPPORTED, "init: FFT length without a plan");
        const char* perr = build_host_plan(lattice, grid, ecut, &c->hp);
        if (perr) return fail(std::strstr(perr, "plan") ? TDDFT_EUNSUPPORTED : TDDFT_EINVAL, std::string("init: ") + perr);
        c->ecut = ecut; c->alpha = alpha; c->nspin = nspin;
        { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev); if (c->num_sms < 1) c->num_sms = 148; }
        c->nocc[0] = nocc[0]; c->nocc[1] = nspin == 2 ? nocc[1] : 0;
        c->psi[0] = psi_up; c->psi[1] = nspin == 2 ? psi_dn : nullptr;
        c->eig_h[0].assign(eig_up, eig_up + nocc[0]);
        if (nspin == 2) c->eig_h[1].assign(eig_dn, eig_dn + nocc[1]);
        if (opt) {
            if (opt->struct_size != (int)sizeof(tddft_options)) return fail(TDDFT_EINVAL, "init: tddft_options.struct_size mismatch");
            if (opt->use_hartree_fxc >= 0) c->use_hartree_fxc = opt->use_hartree_fxc ? 1 : 0;
            if (opt->rho_floor > 0) c->rho_floor = opt->rho_floor;
            c->vloc[0] = opt->vloc_up; c->vloc[1] = nspin == 2 ? opt->vloc_dn : nullptr;
            c->stream = (cudaStream_t)opt->cuda_stream;
            c->workspace_gb = opt->workspace_gb; c->pair_tile = opt->pair_tile; c->fft_batch = opt->fft_batch;
            c->dav_max_subspace = opt->max_subspace; c->dav_max_iter = opt->max_iter; c->dav_tol = opt->tol;
            c->dav_x0 = opt->x0; c->dav_nx0 = opt->n_x0; c->seed = opt->seed;
            c->fused = opt->fft_path == 0;
        } else c->fused = true;
        c->fused = c->fused && fused_supported(grid);
        { const char* e = getenv("TDDFT_CT_FULL"); c->ct_full = !(e && atoi(e) == 0); }
        const long nr = c->hp.nr, npwh = c->hp.npwh;
        if (c->fft_batch <= 0) {
            // large launches win (measured up to 192 grids): with the plane-major unit order the CTAs of a launch share orbital
            // planes whatever its size, and launch tails shrink; up to 96 grids and 640 MB of work grids, among the upper
            // quarter the size whose plane units (n1 per grid) fill whole waves of two CTAs per SM best
            const long cap = std::max<long>(1, std::min<long>(96, (640L << 20) / (16 * nr)));
            const long resident = 2L * c->num_sms;
            long bestb = cap; double beste = 0.0;
            for (long b = cap; b >= std::max<long>(1, cap - cap / 4); --b) {
                int si, sj; choose_subblock((int)(2 * b), &si, &sj);
                const long units = (long)(si * sj + 1) / 2 * grid[0], waves = (units + resident - 1) / resident;   // grids a pair launch really holds
                const double e = (double)units / (double)(waves * resident);
                if (e > beste + 0.01) { beste = e; bestb = b; }
            }
            c->fft_batch = (int)bestb;
        }
#define INIT_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return fail(e_ == cudaErrorMemoryAllocation ? TDDFT_ENOMEM : TDDFT_ECUDA, std::string("init: " #call ": ") + cudaGetErrorString(e_)); } while (0)
        INIT_CUDA(cudaMalloc((void**)&c->d_idx_p, sizeof(int) * npwh));
        INIT_CUDA(cudaMalloc((void**)&c->d_idx_m, sizeof(int) * npwh));
        INIT_CUDA(cudaMalloc((void**)&c->d_kin, sizeof(double) * npwh));
        const std::vector<double>& vc_h = c->fused ? c->hp.vc_c : c->hp.vc;
        const std::vector<int>& idx_p_h = c->fused ? c->hp.idx_p_c : c->hp.idx_p;
        const std::vector<int>& idx_m_h = c->fused ? c->hp.idx_m_c : c->hp.idx_m;
        INIT_CUDA(cudaMalloc((void**)&c->d_vc, sizeof(double) * vc_h.size()));
        if (c->fused) for (int k = 0; k < 2; ++k) {
            INIT_CUDA(cudaMalloc((void**)&c->d_cmap[k], sizeof(int) * c->hp.colmap[k].size()));
            INIT_CUDA(cudaMemcpy(c->d_cmap[k], c->hp.colmap[k].data(), sizeof(int) * c->hp.colmap[k].size(), cudaMemcpyHostToDevice));
        }
        INIT_CUDA(cudaMalloc((void**)&c->d_work, sizeof(cplx) * nr * c->fft_batch));
        INIT_CUDA(cudaMalloc((void**)&c->d_zeros, 1024));
        INIT_CUDA(cudaMemset(c->d_zeros, 0, 1024));
        std::vector<double> kin(npwh);
        for (long g = 0; g < npwh; ++g) kin[g] = 0.5 * c->hp.g2[g];
        INIT_CUDA(cudaMemcpy(c->d_idx_p, idx_p_h.data(), sizeof(int) * npwh, cudaMemcpyHostToDevice));
        INIT_CUDA(cudaMemcpy(c->d_idx_m, idx_m_h.data(), sizeof(int) * npwh, cudaMemcpyHostToDevice));
        INIT_CUDA(cudaMemcpy(c->d_kin, kin.data(), sizeof(double) * npwh, cudaMemcpyHostToDevice));
        INIT_CUDA(cudaMemcpy(c->d_vc, vc_h.data(), sizeof(double) * vc_h.size(), cudaMemcpyHostToDevice));
        for (int a = 0; a < 3; ++a) {
            const int n = grid[a];
            std::vector<cplx> tw(n);
            for (int k = 0; k < n; ++k) {   // exp(-2 pi i k/n), argument reduced exactly, long double sincos
                const long double ang = -2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)n;
                tw[k] = make_double2((double)cosl(ang), (double)sinl(ang));
            }
            INIT_CUDA(cudaMalloc((void**)&c->d_tw[a], sizeof(cplx) * n));
            INIT_CUDA(cudaMemcpy(c->d_tw[a], tw.data(), sizeof(cplx) * n, cudaMemcpyHostToDevice));
        }
        for (int s = 0; s < nspin; ++s) {
            INIT_CUDA(cudaMalloc((void**)&c->d_eig[s], sizeof(double) * c->nocc[s]));
            INIT_CUDA(cudaMemcpy(c->d_eig[s], c->eig_h[s].data(), sizeof(double) * c->nocc[s], cudaMemcpyHostToDevice));
            INIT_CUDA(cudaMalloc((void**)&c->d_phi[s], sizeof(double) * nr * c->nocc[s]));
            FunLayout lay{0, 0, npwh, 1, 0};
            int rc = to_real_space(c, (const cplx*)c->psi[s], lay, c->nocc[s], c->d_phi[s], 0);
            if (rc) { std::string m = c->err; return fail(rc, m); }
        }
        // rho0 and LDA f_xc (Eq. 8)
        for (int a = 0; a < 3; ++a) INIT_CUDA(cudaMalloc((void**)&c->d_fxc[a], sizeof(double) * nr));
        {
            double *ru = nullptr, *rd = nullptr;
            INIT_CUDA(cudaMalloc((void**)&ru, sizeof(double) * nr));
            INIT_CUDA(launch_rho0(c->d_phi[0], c->nocc[0], nr, ru, c->stream));
            if (nspin == 2) { INIT_CUDA(cudaMalloc((void**)&rd, sizeof(double) * nr)); INIT_CUDA(launch_rho0(c->d_phi[1], c->nocc[1], nr, rd, c->stream)); }
            INIT_CUDA(launch_lda_fxc(ru, nspin == 2 ? rd : ru, nr, c->rho_floor, c->d_fxc[0], c->d_fxc[1], c->d_fxc[2], c->stream));
            INIT_CUDA(cudaStreamSynchronize(c->stream));
            cudaFree(ru); cudaFree(rd);
        }
#undef INIT_CUDA
    } catch (const std::bad_alloc&) { return fail(TDDFT_ENOMEM, "init: host allocation failed"); }
    c->stats = tddft_stats{};
    *out = c;
    return TDDFT_OK;
}

int tddft_npw_half(const tddft_ctx* c, long* npwh) { if (!c || !npwh) return TDDFT_EINVAL; *npwh = c->hp.npwh; return TDDFT_OK; }
int tddft_gvectors(const tddft_ctx* c, int* miller) {
    if (!c || !miller) return TDDFT_EINVAL;
    std::memcpy(miller, c->hp.miller.data(), sizeof(int) * 3 * c->hp.npwh);
    return TDDFT_OK;
}
int tddft_vector_len(const tddft_ctx* c, int mode, long* n) {
    if (!c || !n || mode < 0 || mode > 2) return TDDFT_EINVAL;
    const long v = vector_len(c, mode);
    if (v < 0) return TDDFT_EINVAL;
    *n = v; return TDDFT_OK;
}
int tddft_workspace_bytes(const tddft_ctx* c, long long* bytes) { if (!c || !bytes) return TDDFT_EINVAL; *bytes = (long long)c->arena_bytes; return TDDFT_OK; }

int tddft_apply_liouville(tddft_ctx* c, const double* X, double* AX, int nvec, int mode) {
    try { return apply_liouville_dev(c, X, AX, nvec, mode); }
    catch (const std::bad_alloc&) { return set_err(c, TDDFT_ENOMEM, "apply: host allocation failed"); }
}

int tddft_apply_liouville_host(tddft_ctx* c, const double* Xh, double* AXh, int nvec, int mode) {
    if (!c || !Xh || !AXh || nvec < 1 || mode < 0 || mode > 2) return TDDFT_EINVAL;
    const long L = vector_len(c, mode);
    if (L < 0) return set_err(c, TDDFT_EINVAL, "spin flip needs nspin = 2");
    const size_t bytes = sizeof(cplx) * (size_t)L * nvec;
    if (c->host_bytes < bytes) {      // staging buffers are kept between calls (allocation and release of GBs costs milliseconds)
        cudaFree(c->host_dx); cudaFree(c->host_dax); c->host_dx = c->host_dax = nullptr; c->host_bytes = 0;
        if (cudaMalloc((void**)&c->host_dx, bytes) != cudaSuccess || cudaMalloc((void**)&c->host_dax, bytes) != cudaSuccess) {
            cudaGetLastError(); cudaFree(c->host_dx); c->host_dx = nullptr;
            return set_err(c, TDDFT_ENOMEM, "apply_host: device allocation failed");
        }
        c->host_bytes = bytes;
    }
    double *dX = c->host_dx, *dAX = c->host_dax;
    // The spin blocks of a spin-conserving vector are processed one after the other (apply_liouville_dev), so block 1 of X
    // is copied in while block 0 is computed and block 0 of AX is copied out while block 1 is computed: the copies run on
    // their own stream as 2-D copies (nvec rows of one block, pitch = one trial vector), ordered by events.
    const int nblk = (mode == TDDFT_SPIN_CONSERVING) ? c->nspin : 1;
    int rc = TDDFT_OK;
    if (!c->copy_stream) {
        if (cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess) rc = set_err(c, TDDFT_ECUDA, "apply_host: stream creation failed");
        for (int i = 0; i < 2 && !rc; ++i)
            if (cudaEventCreateWithFlags(&c->ev_x_ready[i], cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&c->ev_ax_done[i], cudaEventDisableTiming) != cudaSuccess) rc = set_err(c, TDDFT_ECUDA, "apply_host: event creation failed");
    }
    const size_t pitch = sizeof(cplx) * (size_t)L;
    size_t boff[2] = {0, 0}, bw[2] = {pitch, 0};
    if (nblk == 2) { bw[0] = sizeof(cplx) * (size_t)c->nocc[0] * c->hp.npwh; boff[1] = bw[0]; bw[1] = pitch - bw[0]; }
    cudaEvent_t start = nullptr;
    if (!rc && cudaEventCreateWithFlags(&start, cudaEventDisableTiming) != cudaSuccess) rc = set_err(c, TDDFT_ECUDA, "apply_host: event creation failed");
    if (!rc) {      // the copies start where the caller's stream stands now
        cudaEventRecord(start, c->stream);
        cudaStreamWaitEvent(c->copy_stream, start, 0);
        for (int b = 0; b < nblk && !rc; ++b) {
            if (cudaMemcpy2DAsync((char*)dX + boff[b], pitch, (const char*)Xh + boff[b], pitch, bw[b], nvec, cudaMemcpyHostToDevice, c->copy_stream) != cudaSuccess ||
                cudaEventRecord(c->ev_x_ready[b], c->copy_stream) != cudaSuccess) rc = set_err(c, TDDFT_ECUDA, "apply_host: H2D copy failed");
        }
    }
    if (!rc) {
        c->overlap_copies = true;
        rc = tddft_apply_liouville(c, dX, dAX, nvec, mode);
        c->overlap_copies = false;
    }
    if (!rc) {
        for (int b = 0; b < nblk && !rc; ++b) {
            if (cudaStreamWaitEvent(c->copy_stream, c->ev_ax_done[b], 0) != cudaSuccess ||
                cudaMemcpy2DAsync((char*)AXh + boff[b], pitch, (const char*)dAX + boff[b], pitch, bw[b], nvec, cudaMemcpyDeviceToHost, c->copy_stream) != cudaSuccess)
                rc = set_err(c, TDDFT_ECUDA, "apply_host: D2H copy failed");
        }
        // the caller's stream continues after the last copy
        if (!rc && (cudaEventRecord(start, c->copy_stream) != cudaSuccess || cudaStreamWaitEvent(c->stream, start, 0) != cudaSuccess)) rc = set_err(c, TDDFT_ECUDA, "apply_host: stream join failed");
    }
    if (cudaStreamSynchronize(c->copy_stream) != cudaSuccess && !rc) rc = set_err(c, TDDFT_ECUDA, "apply_host: copy stream failed");
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && !rc) rc = set_err(c, TDDFT_ECUDA, "apply_host: stream failed");
    if (start) cudaEventDestroy(start);
    return rc;
}

int tddft_set_timing(tddft_ctx* c, int enabled) { if (!c) return TDDFT_EINVAL; c->timing = enabled != 0; return TDDFT_OK; }
int tddft_get_stats(const tddft_ctx* c, tddft_stats* out) {
    if (!c || !out) return TDDFT_EINVAL;
    *out = c->stats; out->fft_batch = c->fft_batch; out->fft_path = c->fused ? 0 : 1;
    out->pair_batch = c->last_pair_batch; out->pair_tile = c->last_pair_tile;
    return TDDFT_OK;
}

int tddft_pair_potentials(tddft_ctx* c, int spin, const int* pairs, long n_pairs, double* tau) {
    if (!c || !pairs || !tau || n_pairs < 0 || spin < 0 || spin >= c->nspin) return TDDFT_EINVAL;
    for (long i = 0; i < 2 * n_pairs; ++i) if (pairs[i] < 0 || pairs[i] >= c->nocc[spin]) return set_err(c, TDDFT_EINVAL, "pair index out of range");
    if (n_pairs == 0) return TDDFT_OK;
    int2* d = nullptr;
    TD_CUDA(c, cudaMalloc((void**)&d, sizeof(int2) * n_pairs));
    cudaError_t e = cudaMemcpyAsync(d, pairs, sizeof(int2) * n_pairs, cudaMemcpyHostToDevice, c->stream);
    int rc = (e == cudaSuccess) ? pair_potentials_dev(c, c->d_phi[spin], d, nullptr, n_pairs, 2 * c->fft_batch, tau, 0) : set_err(c, TDDFT_ECUDA, "pair list copy failed");
    cudaStreamSynchronize(c->stream);
    cudaFree(d);
    return rc;
}

int tddft_project(tddft_ctx* c, int spin, double* Y, long nfun) {
    if (!c || !Y || nfun < 1 || spin < 0 || spin >= c->nspin) return TDDFT_EINVAL;
    const size_t cap = project_scratch_doubles(c, c->nocc[spin], (int)nfun, (size_t)1 << 34);
    int rc = ensure_arena(c, sizeof(double) * cap);
    if (rc) return rc;
    return project_rows(c, spin, Y, (int)nfun, (int)nfun, 0, (double*)c->arena, cap);
}

int tddft_gram(tddft_ctx* c, const double* V, const double* W, int m, long n_complex, double* G) {
    if (!c || !V || !W || !G || m < 1 || n_complex < 1) return TDDFT_EINVAL;
    const long K = 2 * n_complex;
    int splits = (int)std::max<long>(1, std::min<long>(1024, K / 8192));
    int rc = ensure_arena(c, sizeof(double) * (size_t)m * m * (splits + 1));
    if (rc) return rc;
    double* part = (double*)c->arena; double* Gd = part + (size_t)m * m * splits;
    TD_CUDA(c, launch_gemm_nt(V, K, W, K, m, 0, Gd, m, m, m, K, 2 * c->hp.npwh, 2.0, splits, part, c->stream));
    TD_CUDA(c, cudaMemcpyAsync(G, Gd, sizeof(double) * m * m, cudaMemcpyDeviceToHost, c->stream));
    TD_CUDA(c, cudaStreamSynchronize(c->stream));
    return TDDFT_OK;
}

int tddft_orbital_real_space(tddft_ctx* c, int spin, int v, double* out) {
    if (!c || !out || spin < 0 || spin >= c->nspin || v < 0 || v >= c->nocc[spin]) return TDDFT_EINVAL;
    TD_CUDA(c, cudaMemcpyAsync(out, c->d_phi[spin] + (long)v * c->hp.nr, sizeof(double) * c->hp.nr, cudaMemcpyDeviceToDevice, c->stream));
    return TDDFT_OK;
}

const char* tddft_last_error(const tddft_ctx* c) { return c ? c->err.c_str() : g_init_error.c_str(); }

#pragma GCC visibility pop
}  // extern "C"
