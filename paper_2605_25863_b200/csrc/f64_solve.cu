// f64_solve.cu -- fp64 partial-pivot solve (placeholder: implemented in a later commit).
#include "linac_internal.h"

extern "C" {
int linac_solve_f64_workspace(int64_t n, int64_t nrhs, size_t* bytes) {
    if (!bytes || n < 0 || nrhs < 0) return LINAC_ERR_INVALID_ARG;
    *bytes = 0;
    return LINAC_OK;
}
int linac_solve_f64(double*, int64_t, int64_t, double*, int64_t, int64_t, double, void*, int64_t*) {
    return LINAC_ERR_INTERNAL;
}
}
