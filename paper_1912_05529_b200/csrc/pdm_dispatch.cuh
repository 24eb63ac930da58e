// pdm_dispatch.cuh -- kernel look-up across translation units.  The unrolled kernel families are
// instantiated in tu_march.cu (three parts), tu_cluster.cu and tu_tiled.cu so that the library
// builds in parallel; pdm_api.cu only asks for function pointers.
#pragma once
#include "kern_march.cuh"
#include "kern_tiled.cuh"
#include "kern_cluster.cuh"
#include "kern_pack.cuh"

#define PDM_R 8
typedef void (*march_fn)(const pdm_march_params);
typedef void (*tiled_fn)(const pdm_tiled_params);
typedef void (*cluster_fn)(const pdm_cluster_params);
typedef void (*pack_fn)(const pdm_pack_params);

// filter half-lengths with a fully unrolled, register-tiled instantiation, in three build parts
#define PDM_L_PART0(X) X(1) X(2) X(3) X(7) X(12)
#define PDM_L_PART1(X) X(15) X(17)
#define PDM_L_PART2(X) X(25)
#define PDM_FOR_EACH_L(X) PDM_L_PART0(X) PDM_L_PART1(X) PDM_L_PART2(X)

// R = outputs per thread: PDM_R, or PDM_R_SMALL for problems with too few warps to fill the SMs
#define PDM_R_SMALL 4
march_fn pdm_march_kernel_part0(int L, bool taps_smem, bool dedup, int R);
march_fn pdm_march_kernel_part1(int L, bool taps_smem, bool dedup, int R);
march_fn pdm_march_kernel_part2(int L, bool taps_smem, bool dedup, int R);
cluster_fn pdm_cluster_kernel_for(int L, bool taps_smem, bool dedup);
tiled_fn pdm_tiled_kernel_for(int L, bool wide, bool alias);
tiled_fn pdm_tiled2_kernel_for(int L, bool wide, bool sym);   // two depth steps per launch, L <= 15

// general (asymmetric-table) builds: R = PDM_R, no row de-duplication / texture share (tu_asym.cu,
// compiled in the same three parts of the filter-length list)
march_fn   pdm_march_kernel_asym_part0(int L, bool taps_smem);
march_fn   pdm_march_kernel_asym_part1(int L, bool taps_smem);
march_fn   pdm_march_kernel_asym_part2(int L, bool taps_smem);
cluster_fn pdm_cluster_kernel_asym_part0(int L, bool taps_smem);
cluster_fn pdm_cluster_kernel_asym_part1(int L, bool taps_smem);
cluster_fn pdm_cluster_kernel_asym_part2(int L, bool taps_smem);
tiled_fn   pdm_tiled_kernel_asym_part0(int L, bool wide);
tiled_fn   pdm_tiled_kernel_asym_part1(int L, bool wide);
tiled_fn   pdm_tiled_kernel_asym_part2(int L, bool wide);
// frequency-packed, temporally blocked x-tiled form (tu_pack.cu, same three parts)
pack_fn    pdm_pack_kernel_part0(int L, bool sym, int threads, bool gtaps);
pack_fn    pdm_pack_kernel_part1(int L, bool sym, int threads, bool gtaps);
pack_fn    pdm_pack_kernel_part2(int L, bool sym, int threads, bool gtaps);
