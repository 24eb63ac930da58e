// tu_tiled.cu -- instantiations of pdm_tiled_step (see pdm_dispatch.cuh).
#include "pdm_dispatch.cuh"

tiled_fn pdm_tiled_kernel_for(int L, bool wide)
{
    switch (L) {
#define X(LL) case LL: return wide ? pdm_tiled_step<LL, PDM_R, 2> : pdm_tiled_step<LL, PDM_R, 1>;
        PDM_FOR_EACH_L(X)
#undef X
    default: return nullptr;
    }
}
