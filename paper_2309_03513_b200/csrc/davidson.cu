// Block Davidson driver -- placeholder until the driver lands in the next commit.
#include "ctx.h"
extern "C" __attribute__((visibility("default"))) int tddft_davidson(tddft_ctx* c, int nroots, int mode, double* evals, double* evecs, int* iters, double* resnorms) {
    (void)nroots; (void)mode; (void)evals; (void)evecs; (void)iters; (void)resnorms;
    return tddft::set_err(c, TDDFT_EUNSUPPORTED, "tddft_davidson: not built yet");
}
