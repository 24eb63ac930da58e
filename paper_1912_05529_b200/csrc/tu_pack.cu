// tu_pack.cu -- instantiations of pdm_pack_kernel (frequency-packed, temporally blocked x-tiled form)
// for one part of the filter-length list (compiled with -DPDM_TU_PART=0/1/2; see pdm_dispatch.cuh).
#include "pdm_dispatch.cuh"

#if PDM_TU_PART == 0
#define PDM_L_THIS(X) PDM_L_PART0(X)
#define PDM_PART_FN pdm_pack_kernel_part0
#elif PDM_TU_PART == 1
#define PDM_L_THIS(X) PDM_L_PART1(X)
#define PDM_PART_FN pdm_pack_kernel_part1
#else
#define PDM_L_THIS(X) PDM_L_PART2(X)
#define PDM_PART_FN pdm_pack_kernel_part2
#endif

template <int NT>
static pack_fn pick(int L, bool sym)
{
    switch (L) {
#define X(LL) case LL: return sym ? pdm_pack_kernel<LL, true, NT> : pdm_pack_kernel<LL, false, NT>;
        PDM_L_THIS(X)
#undef X
    default: return nullptr;
    }
}

// the build that reads tap rows from the global table (256 threads only; see kern_pack.cuh)
static pack_fn pick_gtaps(int L, bool sym)
{
    switch (L) {
#define X(LL) case LL: return sym ? pdm_pack_kernel<LL, true, 256, true> : pdm_pack_kernel<LL, false, 256, true>;
        PDM_L_THIS(X)
#undef X
    default: return nullptr;
    }
}

pack_fn PDM_PART_FN(int L, bool sym, int threads, bool gtaps)
{
    if (gtaps) return threads == 256 ? pick_gtaps(L, sym) : nullptr;
    return threads == 256 ? pick<256>(L, sym) : threads == 384 ? pick<384>(L, sym) : threads == 512 ? pick<512>(L, sym) : nullptr;
}
