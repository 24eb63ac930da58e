// tu_cluster.cu -- instantiations of pdm_cluster_kernel (see pdm_dispatch.cuh).
#include "pdm_dispatch.cuh"

cluster_fn pdm_cluster_kernel_for(int L, bool taps_smem)
{
    switch (L) {
#define X(LL) case LL: return taps_smem ? pdm_cluster_kernel<LL, PDM_R, true> : pdm_cluster_kernel<LL, PDM_R, false>;
        PDM_FOR_EACH_L(X)
#undef X
    default: return nullptr;
    }
}
