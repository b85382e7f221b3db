// Translation unit of the shared-coefficient / complex-RHS kernel (tdma_shared_tma.cuh), kept
// apart from tdma_plan.cu so that the two compile in parallel.
#include "tdma_shared_tma.cuh"

namespace tdma {

bool configure_shared(SharedConfig *out, int nx, int ny, int ncomp, int want_lines, int want_cluster,
                      int want_leaf, int want_slots, int want_ctas, const cudaDeviceProp &prop, const char **why, bool xsweep, bool uniform)
{
    if (!get_encode_tiled()) { *why = "cuTensorMapEncodeTiled not found"; return false; }
    return configure_shared_impl(out, nx, ny, ncomp, want_lines, want_cluster, want_leaf, want_slots, want_ctas, prop, why, xsweep, uniform);
}

cudaError_t launch_shared(SharedConfig &cfg, const SharedArgs &args, cudaStream_t st)
{
    return launch_shared_impl(cfg, args, st);
}

}  // namespace tdma
