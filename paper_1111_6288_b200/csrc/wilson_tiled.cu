// Wilson kernel, variant 2 ("tiled"): placeholder until the shared-memory staged kernel lands.
#include "ov_internal.h"

namespace ov {

bool tiled_supported(const ov_ctx*) { return false; }

int launch_wilson_tiled(ov_ctx* ctx, const double2*, double2*, const Epilogue&) {
    return fail(ctx, OV_EINVAL, "tiled dslash not available");
}

}  // namespace ov
