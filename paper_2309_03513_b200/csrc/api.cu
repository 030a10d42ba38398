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
StageTimer::StageTimer(tddft_ctx* c_, int stage) : c(c_) {
    if (!c->timing) return;
    StageEvent ev; ev.stage = stage;
    cudaEventCreate(&ev.beg); cudaEventCreate(&ev.end);
    cudaEventRecord(ev.beg, c->stream);
    c->events.push_back(ev); idx = (int)c->events.size() - 1;
}
StageTimer::~StageTimer() { if (idx >= 0) cudaEventRecord(c->events[idx].end, c->stream); }
void collect_timing(tddft_ctx* c) {
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
    c->stats.ms_s7_rotate_ace = ms[ST_S7X];
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
static int work_hint(const tddft_ctx* c, int batch, int kind) { return (double)batch * (double)work_stride(c, kind) * sizeof(cplx) > c->work_l2_mb * 1048576.0 ? 1 : 0; }
static SArgs xpass_args(const tddft_ctx* c, int batch, int kind) {
    const int* n = c->hp.n;
    const long inner = c->fused ? c->hp.ncols[kind] : (long)n[1] * n[2];
    SArgs a{}; a.n = n[0]; a.stride = inner; a.inner = inner; a.nouter = 1; a.outer_stride = 0;
    a.nr = work_stride(c, kind); a.batch = batch; a.tw = c->d_tw[0]; a.work = c->d_work; a.ktab = c->d_vc;
    a.whint = work_hint(c, batch, kind);
    return a;
}
static ZArgs zpass_args(const tddft_ctx* c, int batch, int kind) {
    const int* n = c->hp.n;
    ZArgs a{}; a.n = n[2]; a.npencils = (long)n[0] * n[1]; a.nr = c->hp.nr; a.batch = batch; a.tw = c->d_tw[2]; a.tw2 = c->d_tw[1]; a.work = c->d_work;
    a.lscale = 1.0; a.sscale = 1.0;
    a.cmap = c->d_cmap[kind]; a.ncols = c->hp.ncols[kind]; a.wstride = work_stride(c, kind);
    a.whint = work_hint(c, batch, kind); a.cluster = c->prefer_cluster;
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

// tau_p = C[A1[x_p] A2[y_p]] for npairs pairs (device list), two pairs per complex grid.
// d_slots (optional): slot of each pair inside a batch of stot functions; null = slot p.  batch_pairs <= 2*fft_batch pairs per launch.
int pair_potentials_dev(tddft_ctx* c, const double* A1, const double* A2, const int2* d_pairs, const int* d_slots, long npairs,
                        int batch_pairs, double* tau, int chunked, long stot) {
    for (long p0 = 0; p0 < npairs; p0 += batch_pairs) {
        const int np = (int)std::min<long>(batch_pairs, npairs - p0);
        const int nb = (np + 1) / 2;
        ZArgs z = zpass_args(c, nb, KIND_PROD);
        z.phi = A1; z.phi2 = A2; z.pairs = d_pairs + p0; z.npairs = np;
        TD_RC(leg_forward_yz(c, ZL_PAIR, z));
        TD_RC(leg_x(c, SM_CONV, nb, KIND_PROD));
        z.dst = tau; z.nfun = np; z.sscale = 1.0; z.chunked = chunked; z.fbase = d_slots ? 0 : p0; z.ftotal = stot;
        z.slots = d_slots ? d_slots + p0 : nullptr;
        TD_RC(leg_inverse_yz(c, z));
        c->stats.pair_ffts += np;
    }
    return TDDFT_OK;
}

// S1: nfun half-sphere functions -> real space, dst[f][r] = Omega^-1/2 sum_G c_f(G) exp(i G.r)
// The nfun functions are functions fbase0 .. fbase0 + nfun - 1 of a destination batch of ftotal functions (ftotal <= 0: nfun).
int to_real_space(tddft_ctx* c, const cplx* X, FunLayout lay, int nfun, double* dst, int chunked, long fbase0, long ftotal) {
    if (ftotal <= 0) ftotal = nfun;
    const double scale = 1.0 / std::sqrt(c->hp.omega);
    for (int f0 = 0; f0 < nfun; f0 += 2 * c->fft_batch) {
        const int nf = std::min(2 * c->fft_batch, nfun - f0);
        const int nb = (nf + 1) / 2;
        TD_CUDA(c, launch_scatter_pack2(X, lay, f0, nfun, nb, c->d_idx_p, c->d_idx_m, c->d_work, work_stride(c, KIND_SPHERE), c->stream));
        TD_RC(leg_x(c, SM_INV, nb, KIND_SPHERE));
        ZArgs z = zpass_args(c, nb, KIND_SPHERE);
        z.dst = dst; z.nfun = nf; z.sscale = scale; z.chunked = chunked; z.fbase = fbase0 + f0; z.ftotal = ftotal;
        TD_RC(leg_inverse_yz(c, z));
        c->stats.kernel_launches += 1;
    }
    return TDDFT_OK;
}

// S6+S7: real-space functions (chunked batch) -> half sphere, AX = (Omega^1/2/N_r) FFT[src] + (|G|^2/2 - eps_v) X; X = null: no D term
// src: functions fbase0 .. fbase0 + nfun - 1 of a chunked batch of ftotal functions (ftotal <= 0: nfun); accumulate (X == null): AX += result
int to_sphere_plus_d(tddft_ctx* c, const double* src, int nfun, const cplx* X, cplx* AX, FunLayout lay, const double* d_eig, long fbase0, long ftotal,
                     bool accumulate) {
    if (ftotal <= 0) ftotal = nfun;
    const long nr = c->hp.nr;
    const double scale = std::sqrt(c->hp.omega) / (double)nr;
    for (int f0 = 0; f0 < nfun; f0 += 2 * c->fft_batch) {
        const int nf = std::min(2 * c->fft_batch, nfun - f0);
        const int nb = (nf + 1) / 2;
        ZArgs z = zpass_args(c, nb, KIND_SPHERE);
        z.src0 = src; z.src1 = nullptr; z.nfun = nf; z.lscale = 1.0; z.chunked = 1; z.fbase = fbase0 + f0; z.ftotal = ftotal;
        TD_RC(leg_forward_yz(c, ZL_PACK2, z));
        TD_RC(leg_x(c, SM_FWD, nb, KIND_SPHERE));
        TD_CUDA(c, launch_gather_unpack2(c->d_work, work_stride(c, KIND_SPHERE), c->d_idx_p, c->d_idx_m, f0, nfun, nb, scale, X, AX, lay, c->d_kin, d_eig, c->stream, accumulate));
        c->stats.kernel_launches += 1;
    }
    return TDDFT_OK;
}

// S3 Hartree part: vh[kk] = C[scale * (d0[kk] + d1[kk])]
int hartree(tddft_ctx* c, const double* d0, const double* d1, double scale, int kc, double* vh) {
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

// Yout[row] += scale * sum_u basis_u <basis_u|Yin[row]>: two tensor-core GEMMs (S8: P_c of PAPER.md:105; ACE term of D, Eq. 29)
int lowrank_rows(tddft_ctx* c, const double* basis, int nb_, const double* Yin, double* Yout, int nrows, int grp, long grp_stride,
                 double scale, double* O, size_t o_cap) {
    const long k2 = 2 * c->hp.npwh;
    const int no = nb_;
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
    if ((size_t)no * ldo > o_cap) return set_err(c, TDDFT_ENOMEM, "projector scratch too small");
    double* partial = splits > 1 ? O + (size_t)no * ldo : nullptr;
    TD_CUDA(c, launch_gemm_nt(basis, k2, Yin, k2, grp, grp_stride, O, ldo, no, nrows, k2, k2, 2.0, splits, partial, c->stream));
    TD_CUDA(c, launch_gemm_tn_acc(O, ldo, basis, k2, Yout, k2, grp, grp_stride, nrows, k2, no, scale, c->stream));
    c->stats.kernel_launches += 2 + (splits > 1 ? 1 : 0);
    return TDDFT_OK;
}
int project_rows(tddft_ctx* c, int tgt, double* Y, int nrows, int grp, long grp_stride, double* O, size_t o_cap) {
    return lowrank_rows(c, c->psi[tgt], c->nocc[tgt], Y, Y, nrows, grp, grp_stride, -1.0, O, o_cap);
}
size_t project_scratch_doubles(const tddft_ctx* c, int maxocc, int nrows, size_t max_bytes) {
    const size_t one = (size_t)maxocc * ((nrows + 1) & ~1L);
    size_t cap = std::min<size_t>((size_t)1 << 28, max_bytes / 8 / sizeof(double));   // k-split partial sums: <= 2 GB and <= 1/8 of the budget
    int mult = 13;
    while (mult > 1 && one * mult > cap) --mult;
    return one * mult;
}

// ---- real-space orbitals ------------------------------------------------------------------------------
// d_phi[s] <- phi_vs(r), or the rotated phi~_n = sum_v U[v][n] phi_v of Eq. 31 when wannier_u was given (rotation done in the sphere)
static int compute_phi(tddft_ctx* c, int s) {
    const long npwh = c->hp.npwh;
    const int N = c->nocc[s];
    FunLayout lay{0, 0, npwh, 1, 0};
    if (!c->d_U[s]) return to_real_space(c, (const cplx*)c->psi[s], lay, N, c->d_phi[s], 0);
    double* rot = nullptr;
    if (cudaMalloc((void**)&rot, sizeof(cplx) * (size_t)N * npwh) != cudaSuccess) { cudaGetLastError(); return set_err(c, TDDFT_ENOMEM, "rotated orbitals: allocation failed"); }
    cudaError_t e = cudaMemsetAsync(rot, 0, sizeof(cplx) * (size_t)N * npwh, c->stream);
    if (e == cudaSuccess) e = launch_gemm_tn_acc(c->d_U[s], N, c->psi[s], 2 * npwh, rot, 2 * npwh, N, 0, N, 2 * npwh, N, 1.0, c->stream);
    int rc = e == cudaSuccess ? to_real_space(c, (const cplx*)rot, lay, N, c->d_phi[s], 0) : set_err(c, TDDFT_ECUDA, cudaGetErrorString(e));
    cudaStreamSynchronize(c->stream);
    cudaFree(rot);
    return rc;
}
int ensure_phi(tddft_ctx* c, int s) {
    if (!c->phi_shared || c->phi_spin == s) return TDDFT_OK;
    c->phi_spin = -1;
    TD_RC(compute_phi(c, s));
    c->phi_spin = s;
    return TDDFT_OK;
}
// S_mn of Eq. 32 for the exchange orbitals of spin s, HOST S [N][N]
int orbital_overlap(tddft_ctx* c, int s, double* S) {
    const long nr = c->hp.nr;
    const int N = c->nocc[s];
    TD_RC(ensure_phi(c, s));
    double* sq = nullptr;
    const int splits = (int)std::max<long>(1, std::min<long>(64, nr / 16384));
    if (cudaMalloc((void**)&sq, sizeof(double) * ((size_t)N * nr + (size_t)N * N * (splits + 1))) != cudaSuccess) { cudaGetLastError(); return set_err(c, TDDFT_ENOMEM, "overlap: allocation failed"); }
    double* Sd = sq + (size_t)N * nr; double* part = Sd + (size_t)N * N;
    cudaError_t e = launch_square(c->d_phi[s], (long)N * nr, sq, c->stream);
    if (e == cudaSuccess) e = launch_gemm_nt(sq, nr, sq, nr, N, 0, Sd, N, N, N, nr, 0, 1.0, splits, part, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(S, Sd, sizeof(double) * N * N, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(sq);
    if (e != cudaSuccess) return set_err(c, TDDFT_ECUDA, std::string("overlap: ") + cudaGetErrorString(e));
    std::vector<double> d(N);
    for (int m = 0; m < N; ++m) d[m] = std::sqrt(S[(size_t)m * N + m]);
    for (int m = 0; m < N; ++m) for (int n = 0; n < N; ++n) S[(size_t)m * N + n] /= d[m] * d[n];
    return TDDFT_OK;
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
int build_tiles(tddft_ctx* c, int spin, int T, int W) {
    PairTiles& pt = c->tiles[spin];
    const int N = c->nocc[spin];
    if (pt.T == T && pt.W == W && pt.nocc == N && pt.d_pairs) return TDDFT_OK;
    if (pt.d_pairs) cudaFree(pt.d_pairs);
    if (pt.d_pslot) cudaFree(pt.d_pslot);
    pt = PairTiles{};
    pt.T = T; pt.W = W; pt.nocc = N;
    // Processing order: sub-blocks of sbi rows x sbj columns (sbj even, sbi*sbj <= one launch of 2*fft_batch pairs), row-major
    // inside a sub-block.  A launch then multiplies sbi + sbj orbital grids (L2 resident) instead of ~2*fft_batch, and the two
    // pairs packed into one complex grid still share their first orbital.
    choose_subblock(2 * c->fft_batch, &pt.sbi, &pt.sbj);
    pt.batch_pairs = pt.sbi * pt.sbj;
    const std::vector<char>& mask = c->mask[spin];      // near-sightedness truncation (Eq. 32 / explicit pair list); empty = all pairs
    // Tiles: per row block bi the diagonal tile (T x T, packed triangle) and off-diagonal tiles of up to W columns (W a multiple
    // of T chosen from the workspace: a wide tile keeps the row block's accumulators and a[I] in the contraction's registers over
    // more columns, so a[I] / out[I] cross HBM once per W columns instead of once per T).
    const int nb = (N + T - 1) / T;
    std::vector<int2> pairs; std::vector<int> pslot;
    for (int bi = 0; bi < nb; ++bi)
        for (int cj0 = bi * T; cj0 < N; cj0 += (cj0 == bi * T ? T : W)) {
            TileInfo t{};
            t.diag = cj0 == bi * T;
            t.i0 = bi * T; t.ti = std::min(T, N - t.i0); t.j0 = cj0; t.tj = std::min(t.diag ? T : W, N - t.j0);
            t.pair_off = (long)pairs.size();
            // tau slots (the contraction's layout): dense column-major j*ti + i, or the packed upper triangle i(2 tj - i + 1)/2 + (j - i) on the diagonal
            auto slot_of = [&](int i, int j) { return t.diag ? i * (2 * t.tj - i + 1) / 2 + (j - i) : j * t.ti + i; };
            t.nslots = t.diag ? (long)t.ti * (t.ti + 1) / 2 : (long)t.ti * t.tj;
            int cnt = 0;
            for (int si0 = 0; si0 < t.ti; si0 += pt.sbi)
                for (int sj0 = 0; sj0 < t.tj; sj0 += pt.sbj)
                    for (int i = si0; i < std::min(si0 + pt.sbi, t.ti); ++i)
                        for (int j = sj0; j < std::min(sj0 + pt.sbj, t.tj); ++j) {
                            const int gi = t.i0 + i, gj = t.j0 + j;
                            if (gi > gj) continue;
                            if (!mask.empty() && !mask[(size_t)gi * N + gj]) continue;
                            pairs.push_back(make_int2(gi, gj));
                            pslot.push_back(slot_of(i, j));
                            ++cnt;
                        }
            t.npairs = cnt;
            t.partial = cnt < t.nslots;
            pt.max_pairs = std::max<long>(pt.max_pairs, cnt);
            pt.total_pairs += cnt;
            pt.tiles.push_back(t);
        }
    pt.owner.assign(pt.tiles.size(), 0);
    const size_t np = std::max<size_t>(pairs.size(), 1);
    TD_CUDA(c, cudaMalloc((void**)&pt.d_pairs, sizeof(int2) * np));
    TD_CUDA(c, cudaMalloc((void**)&pt.d_pslot, sizeof(int) * np));
    TD_CUDA(c, cudaMemcpyAsync(pt.d_pslot, pslot.data(), sizeof(int) * pslot.size(), cudaMemcpyHostToDevice, c->stream));
    TD_CUDA(c, cudaMemcpyAsync(pt.d_pairs, pairs.data(), sizeof(int2) * pairs.size(), cudaMemcpyHostToDevice, c->stream));
    TD_CUDA(c, cudaStreamSynchronize(c->stream));   // host vectors go out of scope
    return TDDFT_OK;
}

// Sharded apply: the tiles of all spin blocks of the apply are dealt to the shards, heaviest first, each to the least loaded
// shard (the same deterministic list on every shard).
void assign_tile_owners(tddft_ctx* c, const std::vector<int>& spins) {
    if (c->shard_count <= 1) return;
    struct Item { int spin; int idx; long w; };
    std::vector<Item> items;
    for (int sp : spins) { PairTiles& pt = c->tiles[sp]; for (size_t i = 0; i < pt.tiles.size(); ++i) items.push_back({sp, (int)i, (long)pt.tiles[i].npairs}); }
    std::stable_sort(items.begin(), items.end(), [](const Item& x, const Item& y) { return x.w > y.w; });
    std::vector<long> load(c->shard_count, 0);
    for (const Item& it : items) {
        const int r = (int)(std::min_element(load.begin(), load.end()) - load.begin());
        c->tiles[it.spin].owner[it.idx] = r; load[r] += it.w;
    }
}

size_t workspace_budget(const tddft_ctx* c) {
    size_t fr = 0, tot = 0; cudaMemGetInfo(&fr, &tot);
    size_t budget = (size_t)(0.85 * (double)(fr + c->arena_bytes));
    if (c->workspace_gb > 0) budget = std::min(budget, (size_t)(c->workspace_gb * 1073741824.0));
    return budget;
}

// ---- orbital rotation of Eq. 31 in the sphere: dst_n = sum_v U[v][n] src_v for each of kc trial vectors ------
// src rows of trial vector kk at src + kk*src_vstride (doubles), dst likewise; rows are 2*npwh doubles apart.  accumulate = false
// zeroes dst first.  Ut = false uses U[v][n] (to the rotated basis), true uses U^T (back to the canonical basis).
static int rotate_rows(tddft_ctx* c, int spin, bool back, const double* src, long src_vstride, double* dst, long dst_vstride, int kc,
                       bool accumulate) {
    const int N = c->nocc[spin];
    const long k2 = 2 * c->hp.npwh;
    const double* At = back ? c->d_Ut[spin] : c->d_U[spin];     // At[k][m]: forward k = v, m = n: U[v][n]; back k = n, m = v: U^T[n][v]
    for (int kk = 0; kk < kc; ++kk) {
        double* d = dst + (long)kk * dst_vstride;
        if (!accumulate) TD_CUDA(c, cudaMemsetAsync(d, 0, sizeof(double) * k2 * N, c->stream));
        TD_CUDA(c, launch_gemm_tn_acc(At, N, src + (long)kk * src_vstride, k2, d, k2, N, 0, N, k2, N, 1.0, c->stream));
        c->stats.kernel_launches += 1;
    }
    return TDDFT_OK;
}

// ---- one application ------------------------------------------------------------------------------
struct Block { int src, tgt; long off; };   // occupied spin, target spin, offset (complex) inside a trial vector

// ---- one application, streamed plan -------------------------------------------------------------------------------
// Used when a(r) and out(r) of a whole spin block do not fit for all trial vectors (configs 4, 5).  The tile loop is outermost:
// tau of a tile is formed ONCE and the trial vectors are looped inside it, ks at a time; a(r) of the tile's rows and columns is
// recomputed from X for every tile (S1 on (ti + tj)*ks functions) and the tile's contribution to out goes back to the sphere at
// once and is ADDED to AX there (S6 in accumulate mode), so no real-space array is longer than a tile edge.  The extra transforms
// are ~32 (1/ti + 1/tj) per pair FFT (Eq. 6: the pair potentials do not depend on the trial vectors).
static int apply_streamed(tddft_ctx* c, const cplx* X, cplx* AX, int nvec, const std::vector<Block>& blocks, bool hxc, bool sfk, long L, size_t budget) {
    const long nr = c->hp.nr, npwh = c->hp.npwh;
    const int nblk = (int)blocks.size();
    const bool lead = c->shard_rank == 0;
    const size_t grid_b = sizeof(double) * (size_t)chunked_elems(1, nr);
    int maxsrc = 0, maxbasis = 0; bool rot = false;
    for (auto& b : blocks) {
        maxsrc = std::max(maxsrc, c->nocc[b.src]);
        maxbasis = std::max(maxbasis, std::max(c->nocc[b.tgt], c->n_ace[b.tgt]));
        rot = rot || c->d_U[b.src];
    }
    // ---- plan: tile T x W, ks vectors at a time
    const int tcap = contract_full_max_tile(), tpref = contract_full_pref_tile();
    int T = std::min(maxsrc, c->pair_tile > 0 ? std::min(c->pair_tile, tcap) : tpref), ks = nvec, nks = 1;
    size_t fixed = 0;
    auto fixed_bytes = [&]() {
        size_t f = 0;
        if (hxc) f += grid_b * (size_t)nvec * (2 * nblk + 1);
        if (sfk) f += grid_b * (size_t)nvec * 2;
        if (rot) f += 2 * sizeof(cplx) * (size_t)nvec * maxsrc * npwh;
        return f + sizeof(double) * project_scratch_doubles(c, maxbasis, nvec * maxsrc, budget) + 16384;
    };
    fixed = fixed_bytes();
    auto need = [&](int T_, int W_, int ks_) { return fixed + grid_b * ((size_t)T_ * W_ + 2 * (size_t)(T_ + W_) * ks_); };
    // as many vectors together as a tile edge >= 48 allows (tau is formed once either way, but few vectors leave the DMMA tiles of the
    // contraction mostly empty: measured at config 5, 8 vectors at tile 58: S5 15.8 s; 1 vector at tile 72: 98 s), else ever smaller tiles
    {
        const int T0 = T;
        bool found = false;
        for (;;) {
            const int tmin = ks == 1 ? std::min(T0, 2) : std::min(T0, 48);
            for (T = T0; T >= tmin; T -= (T > 16 ? 4 : 1)) if (need(T, T, ks) <= budget) { found = true; break; }
            if (found) break;
            if (ks == 1) return set_err(c, TDDFT_ENOMEM, "workspace budget too small for the streamed plan");
            do { ++nks; } while ((nvec + nks - 1) / nks == ks);
            ks = (nvec + nks - 1) / nks;
        }
    }
    { const int nbk = (maxsrc + T - 1) / T; T = (maxsrc + nbk - 1) / nbk; }
    int W = T;
    while (c->shard_count <= 1 && W < maxsrc - T && need(T, W + T, ks) <= budget && (c->tile_width <= 0 || W + T <= c->tile_width)) W += T;
    int rc = ensure_arena(c, need(T, W, ks));
    if (rc) return rc;
    char* p = c->arena;
    auto carve = [&](size_t bytes) { char* q = p; p += (bytes + 255) / 256 * 256; return (double*)q; };
    double* A = carve(grid_b * (size_t)(T + W) * ks);
    double* O_ = carve(grid_b * (size_t)(T + W) * ks);
    std::vector<double*> drho(nblk, nullptr), V(nblk, nullptr);
    double* vh = nullptr;
    if (hxc) { for (int b = 0; b < nblk; ++b) { drho[b] = carve(grid_b * nvec); V[b] = carve(grid_b * nvec); } vh = carve(grid_b * nvec); }
    if (sfk) { drho[0] = carve(grid_b * nvec); V[0] = carve(grid_b * nvec); }
    cplx *Xr = nullptr, *Yr = nullptr;
    if (rot) { Xr = (cplx*)carve(sizeof(cplx) * (size_t)nvec * maxsrc * npwh); Yr = (cplx*)carve(sizeof(cplx) * (size_t)nvec * maxsrc * npwh); }
    const size_t o_cap = project_scratch_doubles(c, maxbasis, nvec * maxsrc, budget);
    double* Oproj = carve(sizeof(double) * o_cap);
    double* tau = carve(grid_b * (size_t)T * W);
    for (auto& b : blocks) { rc = build_tiles(c, b.src, std::min(T, c->nocc[b.src]), W); if (rc) return rc; }
    { std::vector<int> spins; for (auto& b : blocks) spins.push_back(b.src); assign_tile_owners(c, spins); }
    c->last_pair_tile = T; c->last_tile_width = W; c->last_pair_batch = c->tiles[blocks[0].src].batch_pairs; c->last_kc = ks; c->last_resident = 0;

    if (c->overlap_copies) for (int b = 0; b < nblk; ++b) TD_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_x_ready[b], 0));
    // source of the real-space transforms of block b: X, or the rotated functions of Eq. 31 (one block at a time in Xr)
    auto source = [&](int b, const cplx** src, long* vlen, long* boff) -> int {
        const Block& bl = blocks[b];
        const int no = c->nocc[bl.src];
        if (!c->d_U[bl.src]) { *src = X; *vlen = L; *boff = bl.off; return TDDFT_OK; }
        StageTimer t(c, ST_S7X);
        TD_RC(rotate_rows(c, bl.src, false, (const double*)(X + bl.off), 2 * L, (double*)Xr, 2L * no * npwh, nvec, false));
        *src = Xr; *vlen = (long)no * npwh; *boff = 0;
        return TDDFT_OK;
    };
    // ---- S2 / S3 for all trial vectors: drho by row groups, then the potentials
    if (hxc || sfk) {
        for (int b = 0; b < nblk; ++b) {
            const Block& bl = blocks[b];
            const int no = c->nocc[bl.src];
            TD_RC(ensure_phi(c, bl.src));
            const cplx* src; long vlen, boff;
            TD_RC(source(b, &src, &vlen, &boff));
            for (int g0 = 0; g0 < no; g0 += T + W) {
                const int tg = std::min(T + W, no - g0);
                for (int k0 = 0; k0 < nvec; k0 += ks) {
                    const int kcc = std::min(ks, nvec - k0);
                    { StageTimer t(c, ST_S1);
                      TD_RC(to_real_space(c, src, FunLayout{vlen, boff + (long)g0 * npwh, npwh, kcc, k0}, tg * kcc, A, 1)); }
                    StageTimer t(c, ST_S23);
                    TD_CUDA(c, launch_drho(c->d_phi[bl.src] + (long)g0 * nr, A, tg, kcc, nr, drho[b] + (long)k0 * nr, c->stream, g0 > 0));
                    c->stats.kernel_launches += (kcc + 3) / 4;
                }
            }
        }
        StageTimer t(c, ST_S23);
        if (hxc && c->nspin == 2) {
            rc = hartree(c, drho[0], drho[1], 1.0, nvec, vh); if (rc) return rc;
            TD_CUDA(c, launch_hxc_potential(vh, c->d_fxc[0], drho[0], c->d_fxc[1], drho[1], nvec, nr, V[0], c->stream));
            TD_CUDA(c, launch_hxc_potential(vh, c->d_fxc[1], drho[0], c->d_fxc[2], drho[1], nvec, nr, V[1], c->stream));
            c->stats.kernel_launches += 2;
        } else if (hxc) {
            rc = hartree(c, drho[0], nullptr, 2.0, nvec, vh); if (rc) return rc;
            TD_CUDA(c, launch_hxc_potential(vh, c->d_fxc[0], drho[0], c->d_fxc[1], drho[0], nvec, nr, V[0], c->stream));
            c->stats.kernel_launches += 1;
        } else {
            TD_CUDA(c, launch_scale_potential(c->d_fsf, drho[0], nvec, nr, V[0], c->stream)); c->stats.kernel_launches += 1;
        }
    }
    for (int b = 0; b < nblk; ++b) {
        const Block& bl = blocks[b];
        const int no = c->nocc[bl.src];
        TD_RC(ensure_phi(c, bl.src));
        const double* phi = c->d_phi[bl.src];
        const cplx* src; long vlen, boff;
        TD_RC(source(b, &src, &vlen, &boff));
        const bool rotb = c->d_U[bl.src] != nullptr;
        // destination of the grid part: AX (started from the D term, Eq. 3) or, with the rotation of Eq. 31, Yr (started from zero)
        cplx* dst = rotb ? Yr : AX;
        const long dvlen = rotb ? (long)no * npwh : L, dboff = rotb ? 0 : bl.off;
        FunLayout lay_full{L, bl.off, npwh, nvec, 0};
        auto d_or_zero = [&]() -> int {      // AX block = D X on the lead shard, zero on the others
            if (lead) { TD_CUDA(c, launch_d_term(X, AX, lay_full, no * nvec, c->d_kin, c->d_eig[bl.src], c->stream)); c->stats.kernel_launches += 1; }
            else TD_CUDA(c, cudaMemset2DAsync(AX + bl.off, sizeof(cplx) * L, 0, sizeof(cplx) * (size_t)no * npwh, nvec, c->stream));
            return TDDFT_OK;
        };
        if (rotb) TD_CUDA(c, cudaMemsetAsync(Yr, 0, sizeof(cplx) * (size_t)nvec * no * npwh, c->stream));
        else { StageTimer t(c, ST_S6); TD_RC(d_or_zero()); }
        const double* vloc_b = lead ? c->vloc[bl.tgt] : nullptr;
        const bool has_init = hxc || sfk || vloc_b;
        const PairTiles& pt = c->tiles[bl.src];
        // Row-resident mode (all trial vectors fit at once): the tiles of one row block follow each other (build_tiles), so a[I] is
        // transformed once per row block and out[I] collects the whole row in real space before it goes back to the sphere; only
        // the column side (a[J], out[J]) is per tile.  The batch layout is fixed: rows at functions [0, T*ks), columns from T*ks.
        const bool row_mode = ks == nvec;
        const long ftot_row = (long)(T + W) * ks;
        int row_i0 = -1, row_ti = 0;
        auto flush_row = [&]() -> int {      // S6 of the finished row block
            if (row_i0 < 0) return TDDFT_OK;
            StageTimer tm(c, ST_S6);
            const FunLayout dI{dvlen, dboff + (long)row_i0 * npwh, npwh, ks, 0};
            row_i0 = -1;
            return to_sphere_plus_d(c, O_, row_ti * ks, nullptr, dst, dI, nullptr, 0, ftot_row, true);
        };
        for (size_t tidx = 0; tidx < pt.tiles.size(); ++tidx) {
            const TileInfo& t = pt.tiles[tidx];
            const bool exch = c->alpha != 0.0 && t.npairs > 0 && pt.owner[tidx] == c->shard_rank;
            if (!exch && !(t.diag && has_init)) continue;
            if (exch) {
                StageTimer tm(c, ST_S4);
                if (t.partial) TD_CUDA(c, cudaMemsetAsync(tau, 0, grid_b * (size_t)t.nslots, c->stream));
                rc = pair_potentials_dev(c, phi, phi, pt.d_pairs + t.pair_off, pt.d_pslot + t.pair_off, t.npairs, pt.batch_pairs, tau, 1, t.nslots); if (rc) return rc;
            }
            if (row_mode) {
                const int nI = t.ti * ks, nJ = t.diag ? 0 : t.tj * ks;
                const long fJ = (long)T * ks;
                if (t.i0 != row_i0) {          // a new row block: a[I], and out[I] = phi V + V_loc a (Eq. 4; zero if neither)
                    TD_RC(flush_row());
                    { StageTimer tm(c, ST_S1);
                      TD_RC(to_real_space(c, src, FunLayout{vlen, boff + (long)t.i0 * npwh, npwh, ks, 0}, nI, A, 1, 0, ftot_row)); }
                    StageTimer tm(c, ST_S5);
                    TD_CUDA(c, launch_out_init(phi + (long)t.i0 * nr, (hxc || sfk) ? V[b] : nullptr, vloc_b, A, t.ti, ks, nr, O_, c->stream, ftot_row));
                    c->stats.kernel_launches += 1;
                    row_i0 = t.i0; row_ti = t.ti;
                }
                if (nJ) {
                    { StageTimer tm(c, ST_S1);
                      TD_RC(to_real_space(c, src, FunLayout{vlen, boff + (long)t.j0 * npwh, npwh, ks, 0}, nJ, A, 1, fJ, ftot_row)); }
                    StageTimer tm(c, ST_S5);      // zero the column part of every chunk of out
                    TD_CUDA(c, cudaMemset2DAsync(O_ + fJ * CHUNK, sizeof(double) * ftot_row * CHUNK, 0, sizeof(double) * (size_t)nJ * CHUNK, (size_t)((nr + CHUNK - 1) / CHUNK), c->stream));
                }
                if (exch) {
                    StageTimer tm(c, ST_S5);
                    TD_CUDA(c, launch_contract_full(t.diag, O_, A, tau, 0, t.ti, t.diag ? 0 : T, t.tj, ks, ftot_row, t.nslots, nr, c->alpha, c->stream));
                    c->stats.kernel_launches += (ks + 15) / 16;
                }
                if (nJ) {
                    StageTimer tm(c, ST_S6);
                    TD_RC(to_sphere_plus_d(c, O_, nJ, nullptr, dst, FunLayout{dvlen, dboff + (long)t.j0 * npwh, npwh, ks, 0}, nullptr, fJ, ftot_row, true));
                }
                continue;
            }
            for (int k0 = 0; k0 < nvec; k0 += ks) {
                const int kcc = std::min(ks, nvec - k0);
                const int nI = t.ti * kcc, nJ = t.diag ? 0 : t.tj * kcc;
                const long ftot = nI + nJ;
                const FunLayout layI{vlen, boff + (long)t.i0 * npwh, npwh, kcc, k0}, layJ{vlen, boff + (long)t.j0 * npwh, npwh, kcc, k0};
                { StageTimer tm(c, ST_S1);
                  TD_RC(to_real_space(c, src, layI, nI, A, 1, 0, ftot));
                  if (nJ) TD_RC(to_real_space(c, src, layJ, nJ, A, 1, nI, ftot)); }
                { StageTimer tm(c, ST_S5);
                  if (t.diag) { TD_CUDA(c, launch_out_init(phi + (long)t.i0 * nr, (hxc || sfk) ? V[b] + (long)k0 * nr : nullptr, vloc_b, A, t.ti, kcc, nr, O_, c->stream, ftot)); c->stats.kernel_launches += 1; }
                  else TD_CUDA(c, cudaMemsetAsync(O_, 0, grid_b * (size_t)ftot, c->stream));
                  if (exch) {
                      TD_CUDA(c, launch_contract_full(t.diag, O_, A, tau, 0, t.ti, t.diag ? 0 : t.ti, t.tj, kcc, ftot, t.nslots, nr, c->alpha, c->stream));
                      c->stats.kernel_launches += (kcc + 15) / 16;
                  } }
                StageTimer tm(c, ST_S6);
                const FunLayout dI{dvlen, dboff + (long)t.i0 * npwh, npwh, kcc, k0}, dJ{dvlen, dboff + (long)t.j0 * npwh, npwh, kcc, k0};
                TD_RC(to_sphere_plus_d(c, O_, nI, nullptr, dst, dI, nullptr, 0, ftot, true));
                if (nJ) TD_RC(to_sphere_plus_d(c, O_, nJ, nullptr, dst, dJ, nullptr, nI, ftot, true));
            }
        }
        TD_RC(flush_row());
        if (rotb) {       // Eq. 31: rotate the grid part back and add D
            StageTimer t(c, ST_S7X);
            TD_RC(d_or_zero());
            TD_RC(rotate_rows(c, bl.src, true, (const double*)Yr, 2L * no * npwh, (double*)(AX + bl.off), 2 * L, nvec, true));
        }
        if (lead && c->n_ace[bl.tgt] > 0 && c->alpha != 0.0) {
            StageTimer t(c, ST_S7X);
            rc = lowrank_rows(c, (const double*)c->d_xi[bl.tgt], c->n_ace[bl.tgt], (const double*)(X + bl.off), (double*)(AX + bl.off), nvec * no, no, 2 * L,
                              -c->alpha, Oproj, o_cap);
            if (rc) return rc;
        }
        { StageTimer t(c, ST_S8);
          rc = project_rows(c, bl.tgt, (double*)(AX + bl.off), nvec * no, no, 2 * L, Oproj, o_cap); if (rc) return rc; }
        if (c->overlap_copies) TD_CUDA(c, cudaEventRecord(c->ev_ax_done[b], c->stream));
    }
    collect_timing(c);
    return TDDFT_OK;
}

int apply_liouville_dev(tddft_ctx* c, const double* Xd, double* AXd, int nvec, int mode) {
    if (!c) return TDDFT_EINVAL;
    if (!Xd || !AXd || nvec < 1) return set_err(c, TDDFT_EINVAL, "apply: null buffer or nvec < 1");
    if (Xd == AXd) return set_err(c, TDDFT_EINVAL, "apply: AX must not alias X");
    if (mode < 0 || mode > 2) return set_err(c, TDDFT_EINVAL, "apply: unknown mode");
    if (mode != TDDFT_SPIN_CONSERVING && c->nspin != 2) return set_err(c, TDDFT_EINVAL, "spin flip needs nspin = 2");
    TD_CUDA(c, cudaSetDevice(c->device));
    const cplx* X = (const cplx*)Xd; cplx* AX = (cplx*)AXd;
    const long nr = c->hp.nr, npwh = c->hp.npwh, L = vector_len(c, mode);
    c->stats = tddft_stats{};
    std::vector<Block> blocks;
    if (mode == TDDFT_SPIN_CONSERVING) { long off = 0; for (int s = 0; s < c->nspin; ++s) { blocks.push_back({s, s, off}); off += (long)c->nocc[s] * npwh; } }
    else { const int src = (mode == TDDFT_SPIN_FLIP) ? 0 : 1; blocks.push_back({src, 1 - src, 0}); }
    const int nblk = (int)blocks.size();
    const bool lead = c->shard_rank == 0;      // sharded apply: only shard 0 adds the terms that are not sums over pairs
    const bool hxc = lead && (mode == TDDFT_SPIN_CONSERVING) && c->use_hartree_fxc;
    const bool sfk = lead && (mode != TDDFT_SPIN_CONSERVING) && c->sf_xc;        // K1e^SF of Eq. 24 with the kernel of Eq. 26
    int maxocc = 0, sumsrc = 0, maxsrc = 0, maxbasis = 0;
    bool rot = false;
    for (auto& b : blocks) {
        maxocc = std::max(maxocc, std::max(c->nocc[b.src], c->nocc[b.tgt])); sumsrc += c->nocc[b.src]; maxsrc = std::max(maxsrc, c->nocc[b.src]);
        maxbasis = std::max(maxbasis, std::max(c->nocc[b.tgt], c->n_ace[b.tgt]));
        rot = rot || c->d_U[b.src];
    }

    // ---- workspace plan: all spin blocks resident or one at a time, k chunk kc and tile edge T under the budget ----------------
    const size_t budget = workspace_budget(c);
    const size_t grid_b = sizeof(double) * (size_t)chunked_elems(1, nr);   // one real grid, padded to whole chunks
    const int tcap = contract_full_max_tile(), tpref = contract_full_pref_tile();
    int kc = nvec, T = 0; bool resident = !c->phi_shared; size_t fixed = 0;
    auto fixed_bytes = [&](int kc_, bool res) {
        size_t f = grid_b * (size_t)kc_ * ((size_t)(res ? sumsrc : maxsrc) + (size_t)maxsrc);
        if (hxc) f += grid_b * (size_t)kc_ * (2 * nblk + 1);
        if (sfk) f += grid_b * (size_t)kc_ * 2;
        if (rot) f += 2 * sizeof(cplx) * (size_t)kc_ * maxsrc * npwh;
        return f + sizeof(double) * project_scratch_doubles(c, maxbasis, kc_ * maxsrc, budget) + 8192;
    };
    for (;;) {
        fixed = fixed_bytes(kc, resident);
        T = std::min(maxsrc, c->pair_tile > 0 ? std::min(c->pair_tile, tcap) : tpref);
        const int tmin = std::min(maxsrc, 16);
        while (T > tmin && fixed + grid_b * (size_t)T * T > budget) T = std::max(tmin, T - 4);
        const bool fits = fixed + grid_b * (size_t)T * T <= budget;
        // a small tile costs a(r)/out(r) traffic in S5: before shrinking T below half its cap, give up residency of all blocks
        const int tfloor = c->pair_tile > 0 ? std::min(48, c->pair_tile) : 48;      // an explicitly small pair_tile is the caller's choice
        if (c->plan == 2) { kc = 0; break; }
        if (fits && T >= std::min(maxsrc, std::min(tcap / 2, c->pair_tile > 0 ? c->pair_tile : tcap))) break;
        if (resident && nblk > 1) { resident = false; continue; }
        if (fits && T >= std::min(maxsrc, tfloor)) break;
        if (c->plan == 1) return set_err(c, TDDFT_ENOMEM, "workspace budget too small for the resident plan");
        // a(r) / out(r) of a whole spin block do not fit for all trial vectors: tile loop outermost, tau formed once (apply_streamed)
        kc = 0;
        break;
    }
    if (kc < nvec) return apply_streamed(c, X, AX, nvec, blocks, hxc, sfk, L, budget);      // the vectors do not fit together: tile loop outermost
    if (nblk == 1) resident = true;
    { const int nbk = (maxsrc + T - 1) / T; T = (maxsrc + nbk - 1) / nbk; }   // equal blocks: the kernel's cost follows the largest
    // width of the off-diagonal tiles: as many row blocks as the budget holds (at most what is right of the first row block)
    int W = T;
    while (c->shard_count <= 1 && W < maxsrc - T && fixed + grid_b * (size_t)T * (W + T) <= budget && (c->tile_width <= 0 || W + T <= c->tile_width)) W += T;      // sharded: square tiles, more of them to deal out
    int rc = ensure_arena(c, fixed + grid_b * (size_t)T * W);
    if (rc) return rc;
    char* p = c->arena;
    auto carve = [&](size_t bytes) { char* q = p; p += (bytes + 255) / 256 * 256; return (double*)q; };
    std::vector<double*> a(nblk);
    if (resident) for (int b = 0; b < nblk; ++b) a[b] = carve(grid_b * (size_t)kc * c->nocc[blocks[b].src]);
    else { double* a0 = carve(grid_b * (size_t)kc * maxsrc); for (int b = 0; b < nblk; ++b) a[b] = a0; }
    double* out = carve(grid_b * (size_t)kc * maxsrc);
    std::vector<double*> drho(nblk, nullptr), V(nblk, nullptr);
    double* vh = nullptr;
    if (hxc) { for (int b = 0; b < nblk; ++b) { drho[b] = carve(grid_b * kc); V[b] = carve(grid_b * kc); } vh = carve(grid_b * kc); }
    if (sfk) { drho[0] = carve(grid_b * kc); V[0] = carve(grid_b * kc); }
    cplx *Xr = nullptr, *Yr = nullptr;
    if (rot) { Xr = (cplx*)carve(sizeof(cplx) * (size_t)kc * maxsrc * npwh); Yr = (cplx*)carve(sizeof(cplx) * (size_t)kc * maxsrc * npwh); }
    const size_t o_cap = project_scratch_doubles(c, maxbasis, kc * maxsrc, budget);
    double* O = carve(sizeof(double) * o_cap);
    double* tau = carve(grid_b * (size_t)T * W);
    for (auto& b : blocks) { rc = build_tiles(c, b.src, std::min(T, c->nocc[b.src]), W); if (rc) return rc; }
    { std::vector<int> spins; for (auto& b : blocks) spins.push_back(b.src); assign_tile_owners(c, spins); }
    c->last_pair_tile = T; c->last_tile_width = W; c->last_pair_batch = c->tiles[blocks[0].src].batch_pairs; c->last_kc = kc; c->last_resident = resident ? 1 : 0;

    for (int k0 = 0; k0 < nvec; k0 += kc) {
        const int kcc = std::min(kc, nvec - k0);
        int loaded = -1;                                   // block whose a(r) sits in the shared buffer (non-resident plan)
        // S1: trial functions of block b to real space (rotated to the localized orbitals first if wannier_u was given)
        auto load_block = [&](int b) -> int {
            const Block& bl = blocks[b];
            const int no = c->nocc[bl.src];
            if (c->overlap_copies) TD_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_x_ready[b], 0));     // this block of X has arrived
            TD_RC(ensure_phi(c, bl.src));
            FunLayout lay{L, bl.off, npwh, kcc, k0};
            const cplx* src = X;
            if (c->d_U[bl.src]) {
                StageTimer t(c, ST_S7X);
                TD_RC(rotate_rows(c, bl.src, false, (const double*)(X + (long)k0 * L + bl.off), 2 * L, (double*)Xr, 2L * no * npwh, kcc, false));
                lay = FunLayout{(long)no * npwh, 0, npwh, kcc, 0}; src = Xr;
            }
            StageTimer t(c, ST_S1);
            TD_RC(to_real_space(c, src, lay, no * kcc, a[b], 1));
            loaded = b;
            return TDDFT_OK;
        };
        auto response_density = [&](int b) -> int {      // S2: drho = sum_v phi_v a_v (Eq. 4 inner sum; Eq. 22 for spin flip)
            StageTimer t(c, ST_S23);
            const Block& bl = blocks[b];
            TD_CUDA(c, launch_drho(c->d_phi[bl.src], a[b], c->nocc[bl.src], kcc, nr, drho[b], c->stream));
            c->stats.kernel_launches += (kcc + 3) / 4;
            return TDDFT_OK;
        };
        if (resident) for (int b = 0; b < nblk; ++b) { TD_RC(load_block(b)); if (hxc || sfk) TD_RC(response_density(b)); }
        else if (hxc) for (int b = 0; b < nblk; ++b) { TD_RC(load_block(b)); TD_RC(response_density(b)); }
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
        for (int b = 0; b < nblk; ++b) {
            const Block& bl = blocks[b];
            const int no = c->nocc[bl.src];
            if (!resident && loaded != b) TD_RC(load_block(b));
            TD_RC(ensure_phi(c, bl.src));
            const double* phi = c->d_phi[bl.src];
            if (sfk) {   // K1e^SF: V = f^SF drho^SF (Eq. 24)
                if (!resident) TD_RC(response_density(b));
                StageTimer t(c, ST_S23);
                TD_CUDA(c, launch_scale_potential(c->d_fsf, drho[b], kcc, nr, V[b], c->stream)); c->stats.kernel_launches += 1;
            }
            { StageTimer t(c, ST_S5);
              TD_CUDA(c, launch_out_init(phi, (hxc || sfk) ? V[b] : nullptr, lead ? c->vloc[bl.tgt] : nullptr, a[b], no, kcc, nr, out, c->stream)); c->stats.kernel_launches += 1; }
            // S4 + S5: exact-exchange response, tile by tile (Eq. 6; tau_vv' of PAPER.md:230)
            if (c->alpha != 0.0) {
                const PairTiles& pt = c->tiles[bl.src];
                for (size_t tidx = 0; tidx < pt.tiles.size(); ++tidx) {
                    const TileInfo& t = pt.tiles[tidx];
                    if (t.npairs == 0) continue;            // every pair of the tile was truncated
                    if (pt.owner[tidx] != c->shard_rank) continue;      // another shard's tile
                    { StageTimer tm(c, ST_S4);
                      if (t.partial) TD_CUDA(c, cudaMemsetAsync(tau, 0, grid_b * (size_t)t.nslots, c->stream));
                      rc = pair_potentials_dev(c, phi, phi, pt.d_pairs + t.pair_off, pt.d_pslot + t.pair_off, t.npairs, pt.batch_pairs, tau, 1, t.nslots); if (rc) return rc; }
                    StageTimer tm(c, ST_S5);
                    TD_CUDA(c, launch_contract_full(t.diag, out, a[b], tau, t.i0, t.ti, t.j0, t.tj, kcc, (long)no * kcc, t.nslots, nr, c->alpha, c->stream));
                    c->stats.kernel_launches += (kcc + 15) / 16;
                }
            }
            // S6 + S7: back to the sphere, add D (Eq. 3 with the model H of reading A4)
            FunLayout lay{L, bl.off, npwh, kcc, k0};
            if (c->d_U[bl.src]) {       // Eq. 31: the grid part was computed for the rotated functions, rotate it back and add D
                FunLayout layr{(long)no * npwh, 0, npwh, kcc, 0};
                { StageTimer t(c, ST_S6); rc = to_sphere_plus_d(c, out, no * kcc, nullptr, Yr, layr, nullptr); if (rc) return rc; }
                StageTimer t(c, ST_S7X);
                if (lead) { TD_CUDA(c, launch_d_term(X, AX, lay, no * kcc, c->d_kin, c->d_eig[bl.src], c->stream)); c->stats.kernel_launches += 1; }
                else TD_CUDA(c, cudaMemset2DAsync(AX + (long)k0 * L + bl.off, sizeof(cplx) * L, 0, sizeof(cplx) * (size_t)no * npwh, kcc, c->stream));
                TD_RC(rotate_rows(c, bl.src, true, (const double*)Yr, 2L * no * npwh, (double*)(AX + (long)k0 * L + bl.off), 2 * L, kcc, true));
            } else {
                StageTimer t(c, ST_S6); rc = to_sphere_plus_d(c, out, no * kcc, lead ? X : nullptr, AX, lay, c->d_eig[bl.src]); if (rc) return rc;
            }
            if (lead && c->n_ace[bl.tgt] > 0 && c->alpha != 0.0) {   // H includes alpha V_X^ACE (Eqs. 28-30)
                StageTimer t(c, ST_S7X);
                rc = lowrank_rows(c, (const double*)c->d_xi[bl.tgt], c->n_ace[bl.tgt], (const double*)(X + (long)k0 * L + bl.off),
                                  (double*)(AX + (long)k0 * L + bl.off), kcc * no, no, 2 * L, -c->alpha, O, o_cap);
                if (rc) return rc;
            }
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
    cudaSetDevice(c->device);
    cudaFree(c->d_phi[0]); if (!c->phi_shared) cudaFree(c->d_phi[1]);
    for (int s = 0; s < 2; ++s) { cudaFree(c->d_eig[s]); cudaFree(c->d_U[s]); cudaFree(c->d_Ut[s]); cudaFree(c->d_xi[s]); }
    for (int a = 0; a < 3; ++a) { cudaFree(c->d_tw[a]); cudaFree(c->d_fxc[a]); }
    cudaFree(c->d_work); cudaFree(c->arena); cudaFree(c->d_fsf);
    cudaFree(c->host_dx); cudaFree(c->host_dax);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    for (int i = 0; i < 2; ++i) { if (c->ev_x_ready[i]) cudaEventDestroy(c->ev_x_ready[i]); if (c->ev_ax_done[i]) cudaEventDestroy(c->ev_ax_done[i]); }
    for (int s = 0; s < 2; ++s) { cudaFree(c->tiles[s].d_pairs); cudaFree(c->tiles[s].d_pslot); }
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
        { int dev = 0; cudaGetDevice(&dev); c->device = dev; cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev); if (c->num_sms < 1) c->num_sms = 148; }
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
            c->dav_block = opt->block; c->dav_precond = opt->precond; c->verbose = opt->verbose;
            c->fused = opt->fft_path == 0 || opt->fft_path == 2;
            c->prefer_cluster = opt->fft_path == 2 ? 1 : 0;
            c->tile_width = opt->tile_width;
            if (opt->plan < 0 || opt->plan > 2) return fail(TDDFT_EINVAL, "init: plan must be 0, 1 or 2");
            c->plan = opt->plan;
            if (opt->shard_count > 1) {
                if (opt->shard_rank < 0 || opt->shard_rank >= opt->shard_count) return fail(TDDFT_EINVAL, "init: shard_rank out of range");
                c->shard_rank = opt->shard_rank; c->shard_count = opt->shard_count;
            }
            if (opt->work_l2_mb > 0) c->work_l2_mb = opt->work_l2_mb;
            c->sf_xc = opt->sf_xc_kernel ? 1 : 0; if (opt->sf_cut > 0) c->sf_cut = opt->sf_cut;
            if (c->sf_xc && nspin != 2) return fail(TDDFT_EINVAL, "init: sf_xc_kernel needs nspin = 2");
            if (opt->s_thr < 0 || opt->n_pairs_up < 0 || opt->n_pairs_dn < 0 || opt->n_ace_extra_up < 0 || opt->n_ace_extra_dn < 0)
                return fail(TDDFT_EINVAL, "init: negative s_thr / pair count / ACE orbital count");
            if ((opt->n_ace_extra_up > 0 && !opt->psi_ace_up) || (opt->n_ace_extra_dn > 0 && !opt->psi_ace_dn))
                return fail(TDDFT_EINVAL, "init: n_ace_extra > 0 without psi_ace");
        } else c->fused = true;
        c->fused = c->fused && fused_supported(grid);
        const long nr = c->hp.nr, npwh = c->hp.npwh;
        if (c->fft_batch <= 0) {
            // large launches win (measured up to 192 grids): with the plane-major unit order the CTAs of a launch share orbital
            // planes whatever its size, and launch tails shrink (S4 of NV215-72: 642 / 629 / 628 / 622 / 622 ms at 64 / 90 / 128 /
            // 160 / 192 grids); up to 192 grids and 1.5 GB of work grids, among the upper quarter the size whose plane units
            // (n1 per grid) fill whole waves of two CTAs per SM best
            const long cap = std::max<long>(1, std::min<long>(192, (1536L << 20) / (16 * nr)));
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
        INIT_CUDA(cudaDeviceSynchronize());      // the table uploads above ran on the legacy stream; kernels below run on c->stream
        for (int s = 0; s < nspin; ++s) {
            INIT_CUDA(cudaMalloc((void**)&c->d_eig[s], sizeof(double) * c->nocc[s]));
            INIT_CUDA(cudaMemcpy(c->d_eig[s], c->eig_h[s].data(), sizeof(double) * c->nocc[s], cudaMemcpyHostToDevice));
        }
        // orbital rotation of Eq. 31: U and U^T on the device
        for (int s = 0; s < nspin; ++s) {
            const double* U = opt ? (s == 0 ? opt->wannier_u_up : opt->wannier_u_dn) : nullptr;
            if (!U) continue;
            const int N = c->nocc[s];
            std::vector<double> Ut((size_t)N * N);
            for (int v = 0; v < N; ++v) for (int n = 0; n < N; ++n) Ut[(size_t)n * N + v] = U[(size_t)v * N + n];
            INIT_CUDA(cudaMalloc((void**)&c->d_U[s], sizeof(double) * N * N));
            INIT_CUDA(cudaMalloc((void**)&c->d_Ut[s], sizeof(double) * N * N));
            INIT_CUDA(cudaMemcpy(c->d_U[s], U, sizeof(double) * N * N, cudaMemcpyHostToDevice));
            INIT_CUDA(cudaMemcpy(c->d_Ut[s], Ut.data(), sizeof(double) * N * N, cudaMemcpyHostToDevice));
        }
        // real-space orbitals: one buffer per spin, or one shared buffer refilled on demand when two do not fit comfortably
        {
            size_t fr = 0, tot = 0; cudaMemGetInfo(&fr, &tot);
            const size_t both = sizeof(double) * (size_t)nr * ((size_t)c->nocc[0] + c->nocc[1]);
            c->phi_shared = nspin == 2 && both > (size_t)(0.3 * (double)fr);
            if (c->phi_shared) {
                INIT_CUDA(cudaMalloc((void**)&c->d_phi[0], sizeof(double) * nr * std::max(c->nocc[0], c->nocc[1])));
                c->d_phi[1] = c->d_phi[0];
            } else for (int s = 0; s < nspin; ++s) INIT_CUDA(cudaMalloc((void**)&c->d_phi[s], sizeof(double) * nr * c->nocc[s]));
        }
        // rho0 and LDA f_xc (Eq. 8); spin-flip kernel of Eq. 26
        for (int a = 0; a < 3; ++a) INIT_CUDA(cudaMalloc((void**)&c->d_fxc[a], sizeof(double) * nr));
        {
            double *ru = nullptr, *rd = nullptr;
            INIT_CUDA(cudaMalloc((void**)&ru, sizeof(double) * nr));
            if (nspin == 2) INIT_CUDA(cudaMalloc((void**)&rd, sizeof(double) * nr));
            for (int s = nspin - 1; s >= 0; --s) {          // spin 0 last: a shared buffer then holds the spin the first apply starts with
                c->phi_spin = -1;
                int rc = compute_phi(c, s);
                if (rc) { std::string m = c->err; cudaFree(ru); cudaFree(rd); return fail(rc, m); }
                c->phi_spin = s;
                INIT_CUDA(launch_rho0(c->d_phi[s], c->nocc[s], nr, s == 0 ? ru : rd, c->stream));
            }
            INIT_CUDA(launch_lda_fxc(ru, nspin == 2 ? rd : ru, nr, c->rho_floor, c->d_fxc[0], c->d_fxc[1], c->d_fxc[2], c->stream));
            if (c->sf_xc) {
                INIT_CUDA(cudaMalloc((void**)&c->d_fsf, sizeof(double) * nr));
                INIT_CUDA(launch_sf_kernel_table(ru, rd, nr, c->rho_floor, c->sf_cut, c->d_fsf, c->stream));
            }
            INIT_CUDA(cudaStreamSynchronize(c->stream));
            cudaFree(ru); cudaFree(rd);
        }
        // near-sightedness truncation: explicit pair list, or overlap threshold on Eq. 32
        for (int s = 0; s < nspin; ++s) {
            const int* pl = opt ? (s == 0 ? opt->pair_list_up : opt->pair_list_dn) : nullptr;
            const long np = opt ? (s == 0 ? opt->n_pairs_up : opt->n_pairs_dn) : 0;
            const int N = c->nocc[s];
            if (pl) {
                c->mask[s].assign((size_t)N * N, 0);
                for (long q = 0; q < np; ++q) {
                    const int m = pl[2 * q], n = pl[2 * q + 1];
                    if (m < 0 || n < 0 || m >= N || n >= N) return fail(TDDFT_EINVAL, "init: pair_list index out of range");
                    c->mask[s][(size_t)m * N + n] = 1; c->mask[s][(size_t)n * N + m] = 1;
                }
            } else if (opt && opt->s_thr > 0) {
                std::vector<double> S((size_t)N * N);
                int rc = orbital_overlap(c, s, S.data());
                if (rc) { std::string m = c->err; return fail(rc, m); }
                c->mask[s].assign((size_t)N * N, 0);
                for (size_t e = 0; e < S.size(); ++e) c->mask[s][e] = S[e] >= opt->s_thr ? 1 : 0;
            }
        }
        if (opt && opt->ace) {
            for (int s = 0; s < nspin; ++s) {
                int rc = build_ace(c, s, s == 0 ? opt->psi_ace_up : opt->psi_ace_dn, s == 0 ? opt->n_ace_extra_up : opt->n_ace_extra_dn);
                if (rc) { std::string m = c->err; return fail(rc, m); }
            }
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
    TD_CUDA(c, cudaSetDevice(c->device));
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
    out->pair_batch = c->last_pair_batch; out->pair_tile = c->last_pair_tile; out->tile_width = c->last_tile_width; out->k_chunk = c->last_kc; out->blocks_resident = c->last_resident;
    return TDDFT_OK;
}

int tddft_pair_potentials(tddft_ctx* c, int spin, const int* pairs, long n_pairs, double* tau) {
    if (!c || !pairs || !tau || n_pairs < 0 || spin < 0 || spin >= c->nspin) return TDDFT_EINVAL;
    for (long i = 0; i < 2 * n_pairs; ++i) if (pairs[i] < 0 || pairs[i] >= c->nocc[spin]) return set_err(c, TDDFT_EINVAL, "pair index out of range");
    if (n_pairs == 0) return TDDFT_OK;
    TD_CUDA(c, cudaSetDevice(c->device));
    TD_RC(ensure_phi(c, spin));
    int2* d = nullptr;
    TD_CUDA(c, cudaMalloc((void**)&d, sizeof(int2) * n_pairs));
    cudaError_t e = cudaMemcpyAsync(d, pairs, sizeof(int2) * n_pairs, cudaMemcpyHostToDevice, c->stream);
    int rc = (e == cudaSuccess) ? pair_potentials_dev(c, c->d_phi[spin], c->d_phi[spin], d, nullptr, n_pairs, 2 * c->fft_batch, tau, 0, n_pairs)
                                : set_err(c, TDDFT_ECUDA, "pair list copy failed");
    cudaStreamSynchronize(c->stream);
    cudaFree(d);
    return rc;
}

int tddft_project(tddft_ctx* c, int spin, double* Y, long nfun) {
    if (!c || !Y || nfun < 1 || spin < 0 || spin >= c->nspin) return TDDFT_EINVAL;
    TD_CUDA(c, cudaSetDevice(c->device));
    const size_t cap = project_scratch_doubles(c, c->nocc[spin], (int)nfun, (size_t)1 << 34);
    int rc = ensure_arena(c, sizeof(double) * cap);
    if (rc) return rc;
    return project_rows(c, spin, Y, (int)nfun, (int)nfun, 0, (double*)c->arena, cap);
}

int tddft_gram(tddft_ctx* c, const double* V, const double* W, int m, long n_complex, double* G) {
    if (!c || !V || !W || !G || m < 1 || n_complex < 1) return TDDFT_EINVAL;
    TD_CUDA(c, cudaSetDevice(c->device));
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

int tddft_orbital_overlap(tddft_ctx* c, int spin, double* S) {
    if (!c || !S || spin < 0 || spin >= c->nspin) return TDDFT_EINVAL;
    try { cudaSetDevice(c->device); return orbital_overlap(c, spin, S); }
    catch (const std::bad_alloc&) { return set_err(c, TDDFT_ENOMEM, "overlap: host allocation failed"); }
}

int tddft_orbital_real_space(tddft_ctx* c, int spin, int v, double* out) {
    if (!c || !out || spin < 0 || spin >= c->nspin || v < 0 || v >= c->nocc[spin]) return TDDFT_EINVAL;
    TD_RC(ensure_phi(c, spin));
    TD_CUDA(c, cudaMemcpyAsync(out, c->d_phi[spin] + (long)v * c->hp.nr, sizeof(double) * c->hp.nr, cudaMemcpyDeviceToDevice, c->stream));
    return TDDFT_OK;
}

const char* tddft_last_error(const tddft_ctx* c) { return c ? c->err.c_str() : g_init_error.c_str(); }

#pragma GCC visibility pop
}  // extern "C"
