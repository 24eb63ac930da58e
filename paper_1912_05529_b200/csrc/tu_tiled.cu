// tu_tiled.cu -- instantiations of pdm_tiled_step (see pdm_dispatch.cuh).
#include "pdm_dispatch.cuh"

tiled_fn pdm_tiled_kernel_for(int L, bool wide, bool alias)
{
    if (alias && L == 25) return wide ? pdm_tiled_step<25, PDM_R, 2, true> : pdm_tiled_step<25, PDM_R, 1, true>;
    switch (L) {
#define X(LL) case LL: return wide ? pdm_tiled_step<LL, PDM_R, 2, false> : pdm_tiled_step<LL, PDM_R, 1, false>;
        PDM_FOR_EACH_L(X)
#undef X
    default: return nullptr;
    }
}

// two depth steps per launch: short filters only (halo of at most 2 groups per side)
tiled_fn pdm_tiled2_kernel_for(int L, bool wide, bool sym)
{
    switch (L) {
#define X(LL) case LL: return sym ? (wide ? pdm_tiled_step2<LL, PDM_R, 2, true> : pdm_tiled_step2<LL, PDM_R, 1, true>) \
                                  : (wide ? pdm_tiled_step2<LL, PDM_R, 2, false> : pdm_tiled_step2<LL, PDM_R, 1, false>);
        PDM_L_PART0(X) X(15)
#undef X
    default: return nullptr;
    }
}
