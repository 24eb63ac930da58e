// tu_march.cu -- instantiations of pdm_march_kernel for one part of the filter-length list
// (compiled three times with -DPDM_TU_PART=0/1/2; see pdm_dispatch.cuh).
#include "pdm_dispatch.cuh"

#if PDM_TU_PART == 0
#define PDM_L_THIS(X) PDM_L_PART0(X)
#define PDM_PART_FN pdm_march_kernel_part0
#elif PDM_TU_PART == 1
#define PDM_L_THIS(X) PDM_L_PART1(X)
#define PDM_PART_FN pdm_march_kernel_part1
#else
#define PDM_L_THIS(X) PDM_L_PART2(X)
#define PDM_PART_FN pdm_march_kernel_part2
#endif

template <int RR>
static march_fn pick(int L, bool taps_smem, bool dedup)
{
    switch (L) {
#define X(LL) case LL: return taps_smem ? (dedup ? pdm_march_kernel<LL, RR, true, true> : pdm_march_kernel<LL, RR, true, false>) \
                                         : (dedup ? pdm_march_kernel<LL, RR, false, true> : pdm_march_kernel<LL, RR, false, false>);
        PDM_L_THIS(X)
#undef X
    default: return nullptr;
    }
}

march_fn PDM_PART_FN(int L, bool taps_smem, bool dedup, int R)
{
    return R == PDM_R_SMALL ? pick<PDM_R_SMALL>(L, taps_smem, dedup) : pick<PDM_R>(L, taps_smem, dedup);
}
