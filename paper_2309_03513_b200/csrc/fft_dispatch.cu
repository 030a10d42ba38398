// Routes an FFT length to the translation unit that instantiated it.
#include "common.h"
namespace tddft {
#define TD_DECL(G) \
    cudaError_t launch_zpass_g##G(int, bool, int, int, const ZArgs&, cudaStream_t, bool*); \
    cudaError_t launch_spass_g##G(int, int, const SArgs&, cudaStream_t, bool*);
TD_DECL(0) TD_DECL(1) TD_DECL(2) TD_DECL(3) TD_DECL(4) TD_DECL(5) TD_DECL(6) TD_DECL(7)
#undef TD_DECL

bool fft_size_supported(int n) {
    switch (n) {
#define X(N) case N:
        TD_FOR_EACH_N(X)
#undef X
        return true;
        default: return false;
    }
}
void fft_plan_radices(int n, int* r1, int* r2, int* r3) {
    *r1 = *r2 = *r3 = 0;
    switch (n) {
#define X(N) case N: *r1 = Plan<N>::R1; *r2 = Plan<N>::R2; *r3 = Plan<N>::R3; break;
        TD_FOR_EACH_N(X)
#undef X
        default: break;
    }
}
cudaError_t launch_zpass(bool inverse, int lkind, int skind, const ZArgs& a, cudaStream_t st) {
    bool found = false; cudaError_t e;
#define TRY(G) e = launch_zpass_g##G(a.n, inverse, lkind, skind, a, st, &found); if (found) return e;
    TRY(0) TRY(1) TRY(2) TRY(3) TRY(4) TRY(5) TRY(6) TRY(7)
#undef TRY
    return cudaErrorInvalidValue;
}
cudaError_t launch_spass(int mode, const SArgs& a, cudaStream_t st) {
    bool found = false; cudaError_t e;
#define TRY(G) e = launch_spass_g##G(a.n, mode, a, st, &found); if (found) return e;
    TRY(0) TRY(1) TRY(2) TRY(3) TRY(4) TRY(5) TRY(6) TRY(7)
#undef TRY
    return cudaErrorInvalidValue;
}
}  // namespace tddft
