// K2 tcgen05 path — placeholder until the kernel lands (next commit).
#include "wm_internal.h"

namespace wm {
int tc_prepare(wm_ctx*, const std::vector<std::vector<float>>&, const std::vector<std::string>&) { return WM_OK; }
int tc_supported(const wm_ctx*) { return 0; }
int launch_tc(wm_ctx*, Workspace*, const CallArgs&, cudaStream_t) {
    set_error("tcgen05 path not built");
    return WM_ERR_UNSUPPORTED;
}
}  // namespace wm
