/* tddft.h -- C ABI of the B200-native TDA Liouville (Casida-A) operator of plane-wave hybrid LR-TDDFT
 * (arXiv 2309.03513, "WEST-TDDFT"), Gamma point, real orbitals.
 *
 * The library applies   A = D + K1e - K1d   (Eq. 9; terms: Eq. 3, Eq. 4
 * PAPER.md:82-85, Eq. 6) and its spin-flip counterpart  D^SF - K1d^SF  (PAPER.md:162-182,
 * Eqs. 21, 23, 25) to a block of trial vectors, and finds the lowest roots with a block Davidson solver
 * (PAPER.md:274).  Every step runs in hand-written CUDA kernels for sm_100a; there is no CPU fallback.
 *
 * Conventions:
 *   lattice rows a_i (bohr), Omega = |det A|, reciprocal rows b_i with b_i.a_j = 2 pi delta_ij,
 *   G = m1 b1 + m2 b2 + m3 b3, grid point r_j = sum_i (j_i/n_i) a_i.
 *   Wavefunction sphere |G|^2 <= ecut_wfc_ry (|G|^2 in bohr^-2 equals the kinetic energy in Ry).
 *   Real orbitals: c(-G) = conj c(G); only the canonical HALF sphere is stored: npwh complex coefficients,
 *   G = 0 first with Im c(0) = 0.  phi(r) = Omega^-1/2 sum_G c(G) exp(i G.r), sum_G |c(G)|^2 = 1.
 *   Inner product of half-sphere vectors: <a|b> = 2 Re sum_half conj(a) b - a(0) b(0).
 *   Energies in Hartree, cutoff in Ry.
 *
 * Trial-vector layout (Eq. 2: one function per occupied orbital and spin):
 *   one vector = [spin block][v][g], complex128 interleaved, contiguous; a block of nvec vectors is [k][...].
 *   spin conserving: blocks = spins 0..nspin-1, block s has nocc[s] functions; length = sum_s nocc[s] * npwh
 *   spin flip (up -> down):   one block of nocc[0] functions (occupied-up index v, living in the down space)
 *   spin flip (down -> up):   one block of nocc[1] functions
 *
 * Ownership: the caller owns every buffer.  psi_up/psi_dn (and vloc_*) are BORROWED for the life of the
 * context and must stay valid and unchanged.  The library allocates its own device workspace in tddft_init.
 * Unless stated otherwise pointers named "device" are CUDA device pointers and "host" are host pointers.
 *
 * Errors: every call returns a tddft_status; nothing throws or aborts across the ABI.  CUDA failures give
 * TDDFT_ECUDA with the text available from tddft_last_error.  A context is not thread-safe.
 * All device work is issued on the stream given in tddft_options (default: the legacy default stream).
 * tddft_apply_liouville is asynchronous with respect to the host; tddft_davidson and the *_host variant
 * synchronise the stream before returning.
 */
#ifndef TDDFT_H
#define TDDFT_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tddft_ctx tddft_ctx; /* opaque; one per problem */

typedef enum {
  TDDFT_SPIN_CONSERVING = 0,   /* Eq. 9 */
  TDDFT_SPIN_FLIP = 1,         /* Eq. 21, up occupied -> down virtual: sigma~ = up, sigma = down */
  TDDFT_SPIN_FLIP_DOWN_UP = 2  /* Eq. 21, down occupied -> up virtual */
} tddft_mode;

typedef enum {
  TDDFT_OK = 0,
  TDDFT_EINVAL = 1,        /* bad argument (message in tddft_last_error) */
  TDDFT_ENOMEM = 2,        /* host or device allocation failed */
  TDDFT_ECUDA = 3,         /* a CUDA call or kernel failed */
  TDDFT_ENOTCONVERGED = 4, /* Davidson hit max_iter; outputs hold the best estimates */
  TDDFT_EUNSUPPORTED = 5   /* valid request this build cannot serve (e.g. an FFT length without a plan) */
} tddft_status;

/* All fields optional: pass NULL for defaults, or zero-initialise and set struct_size = sizeof(tddft_options).
 * Pointers are read during tddft_init only, except vloc_* and x0 (borrowed for the life of the context). */
typedef struct {
  int struct_size;          /* ABI versioning: sizeof(tddft_options) of the caller */
  int use_hartree_fxc;      /* spin-conserving K1e (Eq. 4): 1 = on (default), 0 = off; set -1 for "default" */
  double rho_floor;         /* f_xc = 0 where a spin density is below this; <= 0 means default 1e-10 */
  const double* vloc_up;    /* device, [n1*n2*n3] real, optional local potential of the model H (reading A4) */
  const double* vloc_dn;    /* device, idem for spin down (ignored when nspin = 1) */
  void* cuda_stream;        /* cudaStream_t; NULL = legacy default stream */
  double workspace_gb;      /* cap on the library's device workspace; <= 0 = 85 % of free memory at init */
  int pair_tile;            /* orbitals per tile edge T of the exchange loop; <= 0 = chosen from the workspace */
  int fft_batch;            /* packed pair grids per FFT launch; <= 0 = default */
  /* Davidson (reading A11) */
  int max_subspace;         /* <= 0: 12 * nroots */
  int max_iter;             /* <= 0: 200 */
  double tol;               /* residual 2-norm; <= 0: 1e-6 */
  const double* x0;         /* device, n_x0 start vectors in the mode's layout, or NULL: library draws its own */
  int n_x0;
  unsigned long long seed;  /* seed of the library's own start vectors */
  int fft_path;             /* 0 = fused plane/x kernels when the grid shape has them (default), 1 = general pass kernels only,
                             * 2 = fused, with the two-CTA cluster plane kernel wherever the (y,z) plane shape has one */
  int block;                /* Davidson: most correction vectors appended per iteration; <= 0: nroots */
  int precond;              /* Davidson preconditioner: 0 = projector-aware (reading A11b, default), 1 = diagonal */
  int verbose;              /* 1: tddft_davidson prints one line per iteration on stderr */
  /* Spin-flip xc kernel (Eqs. 24, 26; reading A9): 0 = off (default, north star), 1 = on */
  int sf_xc_kernel;
  double sf_cut;            /* f^SF = 0 where |rho_up - rho_dn| < sf_cut (e/bohr^3); <= 0: 1e-3 */
  /* Near-sightedness truncation of K1d (Eqs. 31-32).
   * wannier_u_*: HOST, [nocc][nocc] row-major real orthogonal U with phi_v = sum_n U[v][n] phi~_n; NULL = identity
   *   (the orbitals handed to tddft_init are used as they are).  The real-space part of the operator then runs on the
   *   rotated orbitals phi~ and rotated trial functions a~_n = sum_v U[v][n] a_v, and the result is rotated back.
   * s_thr > 0: pairs (m, n) of (rotated) orbitals with overlap S_mn < s_thr (Eq. 32) are dropped (tau~_mn = 0).
   * pair_list_*: HOST int[2*n_pairs_*], explicit unordered pairs (m, n) to keep; overrides s_thr for that spin;
   *   NULL = all pairs m <= n.  A diagonal pair (m, m) is kept only if listed. */
  const double* wannier_u_up; const double* wannier_u_dn;
  double s_thr;
  const int* pair_list_up; long n_pairs_up;
  const int* pair_list_dn; long n_pairs_dn;
  /* ACE exact exchange inside D (Eqs. 28-30): ace = 1 builds V_X^ACE per spin from the
   * occupied orbitals plus n_ace_extra_* further orbitals (DEVICE complex128 [n_extra][npwh], orthonormal to the
   * occupied ones, read during tddft_init only) and D uses H = T + V_loc + alpha V_X^ACE. */
  int ace;
  const double* psi_ace_up; int n_ace_extra_up;
  const double* psi_ace_dn; int n_ace_extra_dn;
  /* Fused FFT path: launches whose frequency-space work grids are smaller than this many MB leave them to the normal L2
   * replacement policy (they are read back by the next kernel of the pipeline); larger launches stream them with an
   * evict-first hint so that they do not displace the orbital planes.  <= 0: default 48. */
  double work_l2_mb;
  int tile_width;           /* most columns of an off-diagonal tile of the exchange loop (rounded down to a multiple of the tile edge);
                             * <= 0 = as wide as the workspace allows */
  int plan;                 /* memory plan of tddft_apply_liouville: 0 = resident if it fits, else streamed (default); 1 = resident only
                             * (TDDFT_ENOMEM if it does not fit); 2 = streamed (tile loop outermost, pair potentials formed once whatever nvec,
                             * a(r) recomputed per tile, contributions added in the sphere) */
  /* Sharding of ONE apply over several GPUs (the paper's band-group level).  With shard_count > 1 this
   * context applies only the exchange tiles it owns (tiles are dealt to the shards by descending pair count) and only shard 0 adds
   * the terms that are not sums over pairs (D, K1e, V_loc, ACE); every shard projects its partial result (P_c is linear).  The full
   * A X is the SUM of the shards' outputs: one all-reduce of AX, done by the caller (binding.tddft_apply_liouville_sharded uses
   * torch.distributed / NCCL).  Orbitals and X are replicated.  tddft_davidson must not be used with shard_count > 1. */
  int shard_rank;
  int shard_count;
} tddft_options;

/* Canonical half sphere (reading A7 of DESIGN.md): member iff |B^T m|^2 <= ecut_wfc_ry; half = G=0, then m1>0,
 * or m1=0,m2>0, or m1=m2=0,m3>0; ordered by ascending |G|^2 (1e-12 relative ties) then (m1,m2,m3).
 * lattice: host, 9 doubles row-major (rows a1,a2,a3, bohr).  miller: host int[3*capacity] or NULL to query.
 * g2: host double[capacity] or NULL (|G|^2 in bohr^-2).  *npwh receives the count.
 * Returns TDDFT_EINVAL if capacity is too small (count still reported).  Callable before tddft_init. */
int tddft_enumerate_gvectors(const double* lattice, double ecut_wfc_ry, long capacity, int* miller, double* g2,
                             long* npwh);

/* Build a context: G sphere and index maps, Coulomb table 4 pi/|G|^2 (G=0 zeroed),
 * phi_vs(r) for all occupied orbitals, rho0_s = sum_v phi^2 and the LDA f_xc (Eq. 8).
 *   grid:  host int[3], each length must have an FFT plan (2-3-5 smooth, <= 256) and hold the sphere
 *   nspin: 1 (closed shell, singlet channel, reading A6; psi_dn/eig_dn ignored) or 2
 *   nocc:  host int[2]
 *   psi_*: DEVICE complex128 [nocc][npwh], canonical G order, orthonormal (not checked)
 *   eig_*: HOST double[nocc], Hartree
 *   alpha: fraction of exact exchange, >= 0 */
int tddft_init(tddft_ctx** ctx, const double* lattice, const int* grid, double ecut_wfc_ry, int nspin,
               const int* nocc, const double* psi_up, const double* psi_dn, const double* eig_up,
               const double* eig_dn, double alpha, const tddft_options* opt);

int tddft_npw_half(const tddft_ctx* ctx, long* npwh);
/* miller: host int[3*npwh] in canonical order */
int tddft_gvectors(const tddft_ctx* ctx, int* miller);
/* complex elements of one trial vector in the given mode */
int tddft_vector_len(const tddft_ctx* ctx, int mode, long* n_complex);
/* bytes of device workspace the context holds */
int tddft_workspace_bytes(const tddft_ctx* ctx, long long* bytes);

/* AX = A X for a block of nvec trial vectors.  X, AX: DEVICE complex128 [nvec][vector_len],
 * X read-only, AX must not alias X.  The operator projects its output only (Eqs. 3-6 apply P_c on the left). */
int tddft_apply_liouville(tddft_ctx* ctx, const double* X, double* AX, int nvec, int mode);

/* Same with HOST buffers (pinned memory recommended): copies X to the device, applies, copies AX back, synchronises.
 * The copies run on a stream of their own, one spin block at a time, so that a finished block of AX travels back while
 * the next block is still being computed.  Returns after both streams have drained. */
int tddft_apply_liouville_host(tddft_ctx* ctx, const double* X_host, double* AX_host, int nvec, int mode);

/* Lowest nroots of A by block Davidson (reading A11).
 *   evals:    HOST double[nroots], ascending, Hartree
 *   evecs:    DEVICE complex128 [nroots][vector_len] or NULL
 *   iters:    HOST int* or NULL, iterations used
 *   resnorms: HOST double[nroots] or NULL, final residual 2-norms */
int tddft_davidson(tddft_ctx* ctx, int nroots, int mode, double* evals, double* evecs, int* iters,
                   double* resnorms);

/* Off-diagonal block of the full Casida matrix, BX = (K2e - K2d) X (Eq. 1; Eqs. 5, 7 PAPER.md:87-96;
 * SURVEY 8(f)2).  At Gamma with real functions K2e = K1e; K2d is the (phi, a, phi) operand pattern:
 * (K2d X)_v = alpha P_c sum_v' phi_v'(r) C[a_v' phi_v](r), N_occ^2 * nvec pair FFTs.
 * mode = TDDFT_SPIN_CONSERVING: X and BX in the spin-conserving layout.  Spin flip (Eqs. S7, S9): BX is in
 * the layout of `mode`, X is a block of trial vectors of the OPPOSITE flip direction.  X, BX: DEVICE, BX must not alias X.
 * With A X from tddft_apply_liouville the full operator of Eq. 1 is (A X + B Y, B X + A Y). */
int tddft_apply_coupling(tddft_ctx* ctx, const double* X, double* BX, int nvec, int mode);

/* Counters of the last tddft_apply_liouville call (for benchmarks): kernels launched, unique pair potentials
 * tau_vv' formed, and the milliseconds each stage took if timing was enabled. */
typedef struct {
  long long kernel_launches;
  long long pair_ffts;
  double ms_total, ms_s1_to_real, ms_s23_hxc, ms_s4_pair_fft, ms_s5_contract, ms_s6_to_sphere, ms_s8_project;
  double ms_s7_rotate_ace;  /* orbital rotations of Eq. 31 and the ACE term of D */
  int fft_batch; /* packed grids per FFT launch in use */
  int fft_path;  /* 0 = fused plane/x kernels, 1 = general pass kernels */
  int pair_batch; /* orbital pairs per launch of the pair-FFT pipeline in the last apply (<= 2*fft_batch) */
  int pair_tile;  /* tile edge of the last apply */
  int k_chunk;    /* trial vectors processed together (< nvec only under the streamed plan: vectors looped inside a tile) */
  int blocks_resident; /* 1: the real-space functions of all spin blocks were resident; 0: one spin block at a time, or the streamed plan */
  int tile_width;      /* columns of an off-diagonal tile of the last apply (a multiple of pair_tile) */
} tddft_stats;
int tddft_set_timing(tddft_ctx* ctx, int enabled); /* stage timing with CUDA events (adds synchronisation) */
int tddft_get_stats(const tddft_ctx* ctx, tddft_stats* out);

/* Stand-alone pieces of the hot path, exposed for unit parity tests and micro-benchmarks.
 * tddft_pair_potentials: tau_p = C[phi_i phi_j] for n_pairs orbital pairs of one spin;
 *   pairs: HOST int[2*n_pairs]; tau: DEVICE double [n_pairs][n1*n2*n3].
 * tddft_project: Y <- P_c Y on nfun half-sphere functions of target spin `spin`;
 *   Y: DEVICE complex128 [nfun][npwh], in place.
 * tddft_gram: G[i][j] = <V_i|W_j> for m x m full trial vectors; V, W DEVICE [m][n_complex], G HOST. */
int tddft_pair_potentials(tddft_ctx* ctx, int spin, const int* pairs, long n_pairs, double* tau);
int tddft_project(tddft_ctx* ctx, int spin, double* Y, long nfun);
int tddft_gram(tddft_ctx* ctx, const double* V, const double* W, int m, long n_complex, double* G);
/* tddft_gram_static: the same Gram matrix for callers that cannot allocate device memory (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc).  Calls no cudaMalloc / cudaFree / allocating library routine and does not
 * synchronise: the split-k partial sums, which tddft_gram keeps in the context's growable arena, go to a 4 MiB file-scope
 * `static __device__` array that every GPU loading the library holds until exit (gram_static.cu).
 *   V, W: DEVICE complex128 [m][n_complex] as for tddft_gram; G: DEVICE double [m][m], row-major, owned by the caller, valid
 *   once the context's stream has passed the call.  m <= TDDFT_GRAM_STATIC_MAX_M, else TDDFT_EINVAL with a message naming the
 *   limit; the number of k splits shrinks with m so that m * m * splits doubles fit (m <= 22: the splits of tddft_gram, bit-equal
 *   result; larger m: another summation order, equal to rounding).
 *   The array is shared by every context and stream of a device and keeps the last call's partial sums; each call overwrites all
 *   it reads, so nothing is cleared, but two calls that overlap on the GPU (different streams) race on it: keep them ordered.
 *   The first call on a device resolves the array's device address (cudaGetSymbolAddress): make it before a graph capture. */
#define TDDFT_GRAM_STATIC_MAX_M 256
int tddft_gram_static(tddft_ctx* ctx, const double* V, const double* W, int m, long n_complex, double* G);
/* real-space orbital phi_v of a spin on the FFT grid, DEVICE double [n1*n2*n3] out */
int tddft_orbital_real_space(tddft_ctx* ctx, int spin, int v, double* out);
/* Overlap function S_mn of Eq. 32 between the orbitals the exchange term runs on (rotated by
 * wannier_u if given): S HOST double [nocc][nocc]. */
int tddft_orbital_overlap(tddft_ctx* ctx, int spin, double* S);
/* Exact exchange operator on nfun half-sphere functions of one spin (Eq. 28), VY = V_X Y brought back to
 * the sphere: the (phi_occ, psi, phi_occ) operand pattern, nocc * nfun pair FFTs.  use_ace = 1 applies V_X^ACE of Eq. 29
 * instead (needs options.ace).  Y, VY: DEVICE complex128 [nfun][npwh], VY must not alias Y.  No factor alpha. */
int tddft_exchange_apply(tddft_ctx* ctx, int spin, const double* Y, double* VY, long nfun, int use_ace);
/* FP64 peak probes for the roofline denominators (bench.py): register-resident DFMA and DMMA (mma.sync.m8n8k4.f64) loops on
 * every SM, timed with CUDA events on the context's stream.  Both in TFLOP/s, HOST outputs. */
int tddft_fp64_peak(tddft_ctx* ctx, double* dfma_tflops, double* dmma_tflops);
/* Read-bandwidth probe for the access pattern of the exchange contraction (S5): CTAs stream piece_bytes-byte pieces (32, 64, 128 or
 * 256) at a 256-byte stride, 256/piece_bytes CTAs sharing every 256-byte run, over 8 GB.  GB/s, HOST output; CUDA events on the
 * context's stream.  32 is what a contraction CTA (4 grid points of a 32-point chunk) does; 256 is a plain streaming read. */
int tddft_stream_probe(tddft_ctx* ctx, int piece_bytes, double* gbs);

const char* tddft_last_error(const tddft_ctx* ctx); /* ctx may be NULL: error of the last failed tddft_init */
int tddft_destroy(tddft_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* TDDFT_H */
