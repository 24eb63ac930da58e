// kern_cluster.cuh -- PDM_PATH_CLUSTER: the main form with one frequency line split over the CTAs
// of a thread-block cluster (BASELINE.json north_star: "one CTA (or one cluster with DSMEM) holds a
// whole frequency's x-line in shared memory and marches every depth step in place").
//
// CTA `rank` of a cluster of C keeps groups [rank*gper, (rank+1)*gper) of the line (plus HG halo
// groups per side) in its shared memory for all nz steps.  Inside a CTA the depth steps are
// synchronised exactly as in kern_march.cuh (per-warp progress counters between neighbouring
// warps); across CTAs the two edge warps do the same through distributed shared memory:
//   * after step z the first warp PUSHES its first HG output groups into the left neighbour's
//     right-halo slots (and the last warp its last HG groups into the right neighbour's left-halo
//     slots) of the buffer step z+1 will read, then publishes its step count with a
//     release.cluster store into the neighbour's sentinel counter prog[nwarps+1] (resp. prog[0]);
//   * the neighbour's edge warp waits on that sentinel exactly like on a local warp's counter.
// A warp starts step z+1 only when both neighbours have completed step z, which orders both the
// halo read (RAW) and the overwrite of the ping-pong buffer (WAR), as in the single-CTA form.
// Lines are dealt to clusters round-robin (no depth-split hand-off here); two cluster barriers per
// line separate one line's halo pushes from the next line's initialisation.
#pragma once
#include <cooperative_groups.h>
#include "pdm_common.cuh"
#include "kern_march.cuh"

struct pdm_cluster_params {
    const float2 *P0;        // [nw][nx]
    float        *partial;   // [nclusters][nz][pstride]
    const float  *q;         // [nz][qstride]
    const float  *omega;     // [nw]
    const float4 *half;      // [ntab][half16]
    const int    *rowoff;    // [nw+1]
    const int    *rows;      // row lists
    cudaTextureObject_t tex; // the half table as a linear float4 texture
    int nx, nz, nw, ntab;
    int qstride, pstride, half16;
    int ngroups, passes, gper, slots, map_len, nclusters;
    int force_general;       // PDM_FORCE_GENERAL (debug)
};

template <int L, int R, bool TAPS_SMEM, bool DEDUP, bool SYM = true>
__global__ void __launch_bounds__(PDM_MARCH_MAX_THREADS, 1) pdm_cluster_kernel(const pdm_cluster_params p)
{
    namespace cg = cooperative_groups;
    constexpr int HG = pdm_halo_groups<L, R>();
    constexpr int GS = R + 2;
    // per-sample-row plans: row de-duplication and part of the tap gather through the texture unit,
    // exactly as in pdm_march_kernel
    constexpr unsigned TEXMASK = (SYM && DEDUP) ? (L <= 7 ? 0x88u : 0x80u) : 0u;
    cg::cluster_group cluster = cg::this_cluster();
    const int C = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
    const int cid = blockIdx.x / C;

    extern __shared__ __align__(16) unsigned char pdm_smem[];
    float2 *buf_a = reinterpret_cast<float2 *>(pdm_smem);
    float2 *buf_b = buf_a + p.slots;
    unsigned short *map = reinterpret_cast<unsigned short *>(buf_b + p.slots);
    float4 *slice = reinterpret_cast<float4 *>(map + p.map_len);
    __shared__ int prog[PDM_MARCH_MAX_THREADS / 32 + 2];

    const int tid = threadIdx.x, T = blockDim.x;
    const int warp = tid >> 5, lane = tid & 31, nwarps = T >> 5;
    const int ntab_m1 = p.ntab - 1;
    const int gbase = rank * p.gper;                                   // first group of this CTA
    const bool left_active = rank > 0 && gbase < p.ngroups;            // a CTA further left holds groups
    const bool right_active = rank + 1 < C && gbase + p.gper < p.ngroups;
    const int x_lo = gbase * R - HG * R;                               // sample held by slot group 0
    float *const my_partial = p.partial + (size_t)cid * p.nz * p.pstride;
    // remote views of the neighbours' shared memory (same layout in every CTA of the cluster)
    float2 *const lbuf_a = left_active ? cluster.map_shared_rank(buf_a, rank - 1) : buf_a;
    float2 *const rbuf_a = right_active ? cluster.map_shared_rank(buf_a, rank + 1) : buf_a;
    int *const lprog = left_active ? cluster.map_shared_rank(prog, rank - 1) : prog;
    int *const rprog = right_active ? cluster.map_shared_rank(prog, rank + 1) : prog;
    // warps that own at least one group inside the line
    const int npw = min(p.passes, max(0, (p.ngroups - gbase - warp * p.passes * 32 + 31) / 32));

    for (int line = cid; line < p.nw; line += p.nclusters) {
        cluster.sync();                                    // every CTA is done with the previous line
        const float w = p.omega[line];
        if (TAPS_SMEM) {                                   // A2 staging: rows this omega can touch
            const int r0 = p.rowoff[line], nrows = p.rowoff[line + 1] - r0;
            for (int i = tid; i < nrows; i += T) map[p.rows[r0 + i]] = (unsigned short)i;
            const int n4 = nrows * p.half16;
            for (int e = tid; e < n4; e += T) {
                const int s = e / p.half16, c = e - s * p.half16;
                slice[e] = p.half[(size_t)p.rows[r0 + s] * p.half16 + c];
            }
        }
        if (tid < nwarps + 2) {
            bool ahead;                                    // counters that nobody will advance
            if (tid == 0) ahead = !left_active;
            else if (tid == nwarps + 1) ahead = !right_active;
            else ahead = gbase + (tid - 1) * p.passes * 32 >= p.ngroups;
            prog[tid] = ahead ? 0x7fffffff : 0;
        }
        {                                                  // P(0): this CTA's samples and both halos
            const float2 *src = p.P0 + (size_t)line * p.nx;
            const int nslots_g = 2 * HG + p.gper;
            for (int s = tid; s < nslots_g * R; s += T) {
                const int g = s / R, x = x_lo + s;
                float2 v = make_float2(0.f, 0.f);          // R5: zero outside [0,nx)
                if (x >= 0 && x < p.nx) v = __ldcg(src + x);
                buf_a[g * GS + (s - g * R)] = v;
                buf_b[g * GS + (s - g * R)] = make_float2(0.f, 0.f);
            }
        }
        cluster.sync();                                    // initialisation visible before any push

        if (npw > 0) {
            float2 *cur = buf_a, *nxt = buf_b;
            const float4 *const tbase = TAPS_SMEM ? slice : p.half;
            float qn[R];
            int tn[R];
            bool un = false;
            auto load_q = [&](int zq, int pq) {
                const int gq = min(gbase + (warp * p.passes + pq) * 32 + lane, p.ngroups - 1);
                const float4 *qp = reinterpret_cast<const float4 *>(p.q + (size_t)zq * p.qstride + (size_t)gq * R);
#pragma unroll
                for (int i = 0; i < R / 4; ++i) {
                    const float4 v = __ldg(qp + i);
                    qn[4 * i] = v.x; qn[4 * i + 1] = v.y; qn[4 * i + 2] = v.z; qn[4 * i + 3] = v.w;
                }
            };
            auto index_next = [&]() {
                int jn[R];
                bool u = true;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    jn[r] = pdm_index(w, qn[r], ntab_m1);
                    u = u && (jn[r] == jn[0]);
                }
                un = u && !p.force_general;
#pragma unroll
                for (int r = 0; r < R; ++r)
                    tn[r] = (((TEXMASK >> r) & 1u) ? jn[r] : (TAPS_SMEM ? (int)map[jn[r]] : jn[r])) * p.half16;
            };
            load_q(0, 0);
            index_next();
            int qz = 0, qp = 1;
            if (qp == npw) { qp = 0; ++qz; }
            if (qz < p.nz) load_q(qz, qp);
            for (int z = 0; z < p.nz; ++z) {
                const bool accumulate = line >= p.nclusters;           // rows written by an earlier line
                for (int pass = 0; pass < npw; ++pass) {
                    const int gl_raw = (warp * p.passes + pass) * 32 + lane;   // group within this CTA
                    const bool active = gbase + gl_raw < p.ngroups;
                    const int gl = active ? gl_raw : p.ngroups - 1 - gbase;
                    const int g = gbase + gl;                                  // group within the line
                    int toff[R];
#pragma unroll
                    for (int r = 0; r < R; ++r) toff[r] = tn[r];
                    const bool uni = __all_sync(0xffffffffu, un);
                    index_next();
                    if (++qp == npw) { qp = 0; ++qz; }
                    if (qz < p.nz) load_q(qz, qp);
                    float4 *prow = reinterpret_cast<float4 *>(my_partial + (size_t)z * p.pstride + (size_t)g * R);
                    float4 pold[R / 4];
                    if (accumulate) {
#pragma unroll
                        for (int i = 0; i < R / 4; ++i) pold[i] = __ldcs(prow + i);
                    } else {
#pragma unroll
                        for (int i = 0; i < R / 4; ++i) pold[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                    if (pass == 0 && z > 0) {              // A4: both neighbours have completed step z-1
                        if (lane == 0) {
                            int v;
                            do { asm volatile("ld.acquire.cluster.shared.u32 %0, [%1];" : "=r"(v)
                                              : "r"((unsigned)__cvta_generic_to_shared(&prog[warp])) : "memory"); } while (v < z);
                            do { asm volatile("ld.acquire.cluster.shared.u32 %0, [%1];" : "=r"(v)
                                              : "r"((unsigned)__cvta_generic_to_shared(&prog[warp + 2])) : "memory"); } while (v < z);
                        }
                        __syncwarp();
                    }
                    const float2 *base = cur + (HG + gl) * GS;
                    float2 out[R];
                    if (SYM) {
                        if (uni) pdm_fir_group<L, R, true, false>(base, tbase, toff, out);
                        else     pdm_fir_group<L, R, false, DEDUP, TEXMASK>(base, tbase, toff, out, p.tex);
                    } else {
                        if (uni) pdm_fir_group_asym<L, R, true>(base, tbase, toff, out);
                        else     pdm_fir_group_asym<L, R, false>(base, tbase, toff, out);
                    }
                    if (active) {
                        const int x0 = g * R;
                        float2 *dst = nxt + (HG + gl) * GS;
#pragma unroll
                        for (int i = 0; i < R / 2; ++i) {  // samples beyond nx stay zero (R5)
                            float2 a = out[2 * i], b = out[2 * i + 1];
                            if (x0 + 2 * i >= p.nx) a = make_float2(0.f, 0.f);
                            if (x0 + 2 * i + 1 >= p.nx) b = make_float2(0.f, 0.f);
                            *reinterpret_cast<float4 *>(dst + 2 * i) = make_float4(a.x, a.y, b.x, b.y);
                        }
#pragma unroll
                        for (int i = 0; i < R / 4; ++i) {
                            float4 v = pold[i];
                            v.x += out[4 * i].x; v.y += out[4 * i + 1].x;
                            v.z += out[4 * i + 2].x; v.w += out[4 * i + 3].x;
                            __stcs(prow + i, v);
                        }
                    }
                }
                __syncwarp();                              // this warp's step z is in its own shared memory
                // edge warps: copy the HG boundary groups into the neighbour CTA's halo slots of the
                // buffer that step z+1 reads (float4 units: R/2 per group)
                constexpr int N4 = HG * (R / 2);
                if (warp == 0 && left_active) {
                    float2 *rn = lbuf_a + (nxt - buf_a);   // the left CTA's copy of `nxt`
                    for (int i = lane; i < N4; i += 32) {
                        const int gg = i / (R / 2), c = i - gg * (R / 2);
                        *reinterpret_cast<float4 *>(rn + (HG + p.gper + gg) * GS + 2 * c) =
                            *reinterpret_cast<const float4 *>(nxt + (HG + gg) * GS + 2 * c);
                    }
                }
                if (warp == nwarps - 1 && right_active) {
                    float2 *rn = rbuf_a + (nxt - buf_a);
                    for (int i = lane; i < N4; i += 32) {
                        const int gg = i / (R / 2), c = i - gg * (R / 2);
                        *reinterpret_cast<float4 *>(rn + gg * GS + 2 * c) =
                            *reinterpret_cast<const float4 *>(nxt + (p.gper + gg) * GS + 2 * c);
                    }
                }
                // only the two edge warps wrote into another CTA: the cluster-scope fence (which also
                // invalidates L1) is theirs alone, interior warps order their step with a CTA fence
                if ((warp == 0 && left_active) || (warp == nwarps - 1 && right_active))
                    asm volatile("fence.acq_rel.cluster;" ::: "memory");
                else
                    __threadfence_block();
                __syncwarp();
                if (lane == 0) {                           // A4: publish this warp's step z
                    const int done = z + 1;
                    *(volatile int *)&prog[warp + 1] = done;
                    if (warp == 0 && left_active)
                        asm volatile("st.release.cluster.u32 [%0], %1;" :: "l"(lprog + nwarps + 1), "r"(done) : "memory");
                    if (warp == nwarps - 1 && right_active)
                        asm volatile("st.release.cluster.u32 [%0], %1;" :: "l"(rprog), "r"(done) : "memory");
                }
                float2 *t = cur; cur = nxt; nxt = t;
            }
        }
    }
    cluster.sync();                                        // no CTA exits while a neighbour may still push to it
}
