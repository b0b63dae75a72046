// shd_min.cu -- step a5 (on-device minimizer).  Placeholder until the evaluation path is verified.
#include "../../include/shd.h"
#include "shd_internal.h"

void shd_min_free(shd_ctx*) {}

extern "C" int shd_minimize(shd_ctx* h, double*, double*, const shd_min_opts*, shd_min_report*) {
    if (h) h->err = "shd_minimize: not built yet";
    return SHD_EINVAL;
}
