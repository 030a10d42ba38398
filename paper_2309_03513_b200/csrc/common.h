// Shared declarations of the tddft_b200 library (host side).  Product code: no oracle, no CPU fallback.
#pragma once
#include <cuda_runtime.h>
#include <string>
#include <vector>
#include "../../include/tddft.h"
#include "fft_core.cuh"

namespace tddft {

// Per-device caches of function attributes and occupancy (one process may hold contexts on several GPUs): index = device id.
constexpr int kMaxDevices = 64;
inline int current_device() { int d = 0; cudaGetDevice(&d); return (d >= 0 && d < kMaxDevices) ? d : 0; }

// ---- FFT pass launchers (fft_inst.cu; one translation unit per size group) ---------------------------
enum ZLoadKind { ZL_WORK = 0, ZL_PAIR = 1, ZL_PACK2 = 2 };
enum ZStoreKind { ZS_WORK = 0, ZS_SPLIT2 = 1 };

struct ZArgs {
    // geometry
    int n;                 // length of the contiguous axis
    long npencils;         // pencils per grid (n1*n2)
    long nr;               // points per grid
    int batch;             // packed grids in this launch
    const cplx* tw;        // device twiddles exp(-2 pi i k/n)
    const cplx* tw2;       // fused plane kernels only: twiddles of the y axis
    cplx* work;            // [batch][nr] complex work grids (source for ZL_WORK, destination for ZS_WORK)
    // ZL_PAIR: packed grid b = phi[pairs[2b].x]*phi[pairs[2b].y] + i phi[pairs[2b+1].x]*phi[pairs[2b+1].y]
    const double* phi;     // [norb][nr]
    const double* phi2;    // second operand array of the pair products, plain [nfun][nr]; null = phi (pairs of orbitals)
    const int2* pairs;     // device, npairs entries (already offset to this launch)
    int npairs;
    // ZL_PACK2: re = scale*(src0[2b] + src1[2b]), im = same for 2b+1 (src1 optional); nfun functions
    const double* src0;
    const double* src1;
    double lscale;
    // ZS_SPLIT2: dst[2b] = sscale*re, dst[2b+1] = sscale*im  (nfun functions; pairs mode uses npairs)
    double* dst;
    int nfun;
    double sscale;
    const int* slots;      // optional (device, already offset to this launch): function index of packed function q is slots[q]
    // layout of the real function batches src0/src1/dst: function index fbase + (0..nfun-1) inside a batch of ftotal
    // functions; chunked = 0: [f][nr];  chunked = 1: [nr/CHUNK][ftotal][CHUNK] (CHUNK consecutive grid points per function)
    int chunked; long fbase; long ftotal;
    // fused path only: pruned layout of the work grids (plan.h): column map, live columns, grid stride in `work`
    const int* cmap; int ncols; long wstride;
    int whint;             // L2 policy of the work-grid stream: 1 = evict first, 0 = normal (the launch's work grids fit in L2)
    int cluster;           // prefer the two-CTA cluster plane kernel (fft_cluster.cuh) where the shape has both variants
};
// Chunked layout of real-space function batches: [nr/CHUNK][function][CHUNK].  The plane kernels write CHUNK consecutive points
// of a function as one run and a CTA of the contraction (contract.cu) reads 4 points (32 bytes) of every function.  Measured at
// config 3 (block apply, S4 + S5 ms): CHUNK 32: 627 + 320; 16: 640 + 322; 8: 655 + 297; 4: 689 + 266 -- what the contraction gains
// from longer runs of its own the pair-FFT pipeline loses on its stores, the sum stays within 1 %; 32 is kept.
constexpr int CHUNK_LOG = 5;
constexpr int CHUNK = 1 << CHUNK_LOG;
inline long chunked_elems(long nfun, long nr) { return (nr + CHUNK - 1) / CHUNK * CHUNK * nfun; }
// strided passes along an axis with element stride `stride` over `inner` contiguous elements, `nouter` slabs
enum SMode { SM_FWD = 0, SM_INV = 1, SM_CONV = 2 /* forward, multiply by ktab, inverse */ };
struct SArgs {
    int n; long stride; long inner; long nouter; long outer_stride; long nr; int batch;
    const cplx* tw; cplx* work; const double* ktab;   // ktab [nr] real, same (scrambled) layout as work
    int whint;             // fused path: L2 policy of the work-grid stream (see ZArgs)
};
bool fft_size_supported(int n);
cudaError_t launch_zpass(bool inverse, int lkind, int skind, const ZArgs& a, cudaStream_t st);
cudaError_t launch_spass(int mode, const SArgs& a, cudaStream_t st);
void fft_plan_radices(int n, int* r1, int* r2, int* r3);   // 0s if unsupported
// fused fast path (fft_fused.cu): y+z transforms of one x-plane per CTA, register-resident x pass
bool fused_supported(const int* n);
cudaError_t launch_plane(int ny, int nz, bool inverse, int lkind, int skind, const ZArgs& a, cudaStream_t st);
cudaError_t launch_xpass(int mode, const SArgs& a, cudaStream_t st);

}  // namespace tddft
