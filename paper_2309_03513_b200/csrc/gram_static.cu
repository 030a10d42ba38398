// tddft_gram_static: the Davidson Gram matrix G[i][j] = <V_i|W_j> (the Rayleigh-Ritz step of the block Davidson
// solver around Eq. 1) for callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving
// loops, harnesses that forbid allocation.  Same split-k DMMA kernels as tddft_gram (gemm.cu: launch_gemm_nt); what differs is
// where the per-split partial sums live: not in the context's arena (api.cu: ensure_arena may cudaMalloc) but in the file-scope
// device array below, which every GPU that loads the library holds until exit.
//
//   scratch  : kScratchDoubles doubles = 4 MiB, 256-byte aligned, partial[split][m][m]
//   limit    : m <= TDDFT_GRAM_STATIC_MAX_M (256); the k splits are cut down to what fits (m <= 22 keeps all 1024)
//   contents : every call overwrites the partial sums it later reads (each split writes its whole m x m block), so nothing has
//              to start at zero; the array keeps the last call's partial sums
//   sharing  : ONE array per device for every context and stream: calls that overlap on the GPU race on it
//
// In host code `g_gram_scratch` is a host-side stand-in, not a device address; the address the kernels get comes from
// cudaGetSymbolAddress, resolved once per device with that device current (scratch_on_device).
#include <algorithm>
#include <mutex>
#include <string>
#include "ctx.h"

using namespace tddft;

namespace {

constexpr long kScratchDoubles = 1L << 19;   // 4 MiB
static __device__ __align__(256) double g_gram_scratch[kScratchDoubles];

std::mutex g_scratch_mu;
double* g_scratch_ptr[kMaxDevices] = {nullptr};

// device address of g_gram_scratch on `dev`, which must be the current device
cudaError_t scratch_on_device(int dev, double** out) {
    std::lock_guard<std::mutex> lock(g_scratch_mu);
    if (!g_scratch_ptr[dev]) {
        double* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void**)&p, g_gram_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" {
#pragma GCC visibility push(default)

int tddft_gram_static(tddft_ctx* c, const double* V, const double* W, int m, long n_complex, double* G) {
    if (!c || !V || !W || !G || m < 1 || n_complex < 1) return TDDFT_EINVAL;
    if (m > TDDFT_GRAM_STATIC_MAX_M)
        return set_err(c, TDDFT_EINVAL, "gram_static: m = " + std::to_string(m) + " exceeds the static scratch limit of " +
                                            std::to_string(TDDFT_GRAM_STATIC_MAX_M) + " vectors (4 MiB of partial sums); use tddft_gram");
    if (c->device < 0 || c->device >= kMaxDevices) return set_err(c, TDDFT_EINVAL, "gram_static: device ordinal out of range");
    TD_CUDA(c, cudaSetDevice(c->device));
    double* part = nullptr;
    TD_CUDA(c, scratch_on_device(c->device, &part));
    const long K = 2 * n_complex, mm = (long)m * m;
    // tddft_gram's split count, cut down to the scratch: kScratchDoubles / mm >= 8 for every m within the limit
    const int splits = (int)std::max<long>(1, std::min<long>(std::min<long>(1024, K / 8192), kScratchDoubles / mm));
    TD_CUDA(c, launch_gemm_nt(V, K, W, K, m, 0, G, m, m, m, K, 2 * c->hp.npwh, 2.0, splits, part, c->stream));
    return TDDFT_OK;
}

#pragma GCC visibility pop
}  // extern "C"
