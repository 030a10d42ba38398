// Instantiations of the FFT pass kernels for one group of sizes (TD_GROUP = 0..TD_NGROUPS-1), so that the
// groups compile in parallel.  fft_dispatch.cu routes a length to its group.
#include "fft_steps.cuh"
#ifndef TD_GROUP
#error "compile with -DTD_GROUP=k"
#endif
namespace tddft {

#if TD_GROUP == 0
#define TD_SIZES(X) X(4) X(5) X(6) X(8) X(9) X(10) X(12) X(15) X(16) X(18) X(20)
#elif TD_GROUP == 1
#define TD_SIZES(X) X(24) X(25) X(27) X(30) X(32) X(36)
#elif TD_GROUP == 2
#define TD_SIZES(X) X(40) X(45) X(48) X(50) X(54)
#elif TD_GROUP == 3
#define TD_SIZES(X) X(60) X(64) X(72) X(75)
#elif TD_GROUP == 4
#define TD_SIZES(X) X(80) X(81) X(90) X(96)
#elif TD_GROUP == 5
#define TD_SIZES(X) X(100) X(108) X(120) X(125)
#elif TD_GROUP == 6
#define TD_SIZES(X) X(128) X(144) X(150) X(160) X(180)
#elif TD_GROUP == 7
#define TD_SIZES(X) X(192) X(200) X(216) X(240) X(250) X(256)
#endif

#define TD_CAT2(a, b) a##b
#define TD_CAT(a, b) TD_CAT2(a, b)

cudaError_t TD_CAT(launch_zpass_g, TD_GROUP)(int n, bool inverse, int lkind, int skind, const ZArgs& a, cudaStream_t st, bool* found) {
    *found = true;
    switch (n) {
#define X(N) case N: return zpass_dispatch<N>(inverse, lkind, skind, a, st);
        TD_SIZES(X)
#undef X
        default: *found = false; return cudaSuccess;
    }
}
cudaError_t TD_CAT(launch_spass_g, TD_GROUP)(int n, int mode, const SArgs& a, cudaStream_t st, bool* found) {
    *found = true;
    switch (n) {
#define X(N) case N: return spass_dispatch<N>(mode, a, st);
        TD_SIZES(X)
#undef X
        default: *found = false; return cudaSuccess;
    }
}
}  // namespace tddft
