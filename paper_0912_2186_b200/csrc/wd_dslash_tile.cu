// wd_dslash_tile.cu -- WD_KERNEL_TILE (placeholder until the shared-memory kernel lands).
#include "wd_internal.h"

namespace wd {

bool tile_supported(const ApplyArgs &) { return false; }
cudaError_t launch_tile(const ApplyArgs &) { return cudaErrorNotSupported; }

} // namespace wd
