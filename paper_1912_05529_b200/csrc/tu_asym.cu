// tu_asym.cu -- instantiations of the three kernel forms for tables that are not symmetric in k
// (pdm_fir_group_asym), for one part of the filter-length list
// (compiled three times with -DPDM_TU_PART=0/1/2; see pdm_dispatch.cuh).
#include "pdm_dispatch.cuh"

#if PDM_TU_PART == 0
#define PDM_L_THIS(X) PDM_L_PART0(X)
#define PDM_FN(name) name##_part0
#elif PDM_TU_PART == 1
#define PDM_L_THIS(X) PDM_L_PART1(X)
#define PDM_FN(name) name##_part1
#else
#define PDM_L_THIS(X) PDM_L_PART2(X)
#define PDM_FN(name) name##_part2
#endif

march_fn PDM_FN(pdm_march_kernel_asym)(int L, bool taps_smem)
{
    switch (L) {
#define X(LL) case LL: return taps_smem ? pdm_march_kernel<LL, PDM_R, true, false, false> \
                                         : pdm_march_kernel<LL, PDM_R, false, false, false>;
        PDM_L_THIS(X)
#undef X
    default: return nullptr;
    }
}

cluster_fn PDM_FN(pdm_cluster_kernel_asym)(int L, bool taps_smem)
{
    switch (L) {
#define X(LL) case LL: return taps_smem ? pdm_cluster_kernel<LL, PDM_R, true, false, false> \
                                         : pdm_cluster_kernel<LL, PDM_R, false, false, false>;
        PDM_L_THIS(X)
#undef X
    default: return nullptr;
    }
}

tiled_fn PDM_FN(pdm_tiled_kernel_asym)(int L, bool wide)
{
    switch (L) {
#define X(LL) case LL: return wide ? pdm_tiled_step<LL, PDM_R, 2, false, false> \
                                    : pdm_tiled_step<LL, PDM_R, 1, false, false>;
        PDM_L_THIS(X)
#undef X
    default: return nullptr;
    }
}
