// tu_cluster.cu -- instantiations of pdm_cluster_kernel (see pdm_dispatch.cuh).
#include "pdm_dispatch.cuh"

cluster_fn pdm_cluster_kernel_for(int L, bool taps_smem, bool dedup)
{
    switch (L) {
#define X(LL) case LL: return taps_smem ? (dedup ? pdm_cluster_kernel<LL, PDM_R, true, true> : pdm_cluster_kernel<LL, PDM_R, true, false>) \
                                         : (dedup ? pdm_cluster_kernel<LL, PDM_R, false, true> : pdm_cluster_kernel<LL, PDM_R, false, false>);
        PDM_FOR_EACH_L(X)
#undef X
    default: return nullptr;
    }
}
