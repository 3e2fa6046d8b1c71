// Stage 3 + the MLP half of stage 4 as ONE persistent kernel (tensor-core modes): a CTA owns a 128-atom row tile and
// takes it through the whole chain  G -> h1 -> h2 -> h3 (-> e_i, delta3) -> delta2 -> delta1 -> dE/dG  without leaving
// the SM (ChemicalNet; forces by reverse mode, L65 / L176; the model of Fig. 2 is one fused executable,
// L176).  SURVEY.md 8(f)-4 / 8(d) "intermediates": the unfused path (mlp_tc.cu, six launches) writes and re-reads every
// activation through HBM (~0.8 GB per step on the 98k water box) and pays six launch / pipeline-fill costs.
//
// How a layer feeds the next one.  The accumulator of GEMM j lives in TMEM ([128 atoms] x [N_j columns], fp32).  When its
// last MMA has completed, the epilogue warps drain it 16 columns at a time: bias + CELU (forward) or x CELU'(h) (reverse),
// split into tf32 hi / lo, and write the two 128 x 16 blocks back into TMEM as an A-operand "slot" (tcgen05.st).  The MMA
// thread multiplies each slot with the matching 16 rows of W_{j+1} as soon as it is ready (tcgen05.mma .ts form: A from
// TMEM, B = weight tile in shared memory), so GEMM j+1 runs while the epilogue of GEMM j is still producing its operand.
// Nothing but the weights is streamed: they are pre-packed at set-up into the exact 128-byte-swizzled K-major tile images
// the MMA descriptors expect ([K block of 32][part][hi | lo][rows][32]), so one tile is one contiguous cp.async.bulk of
// up to 32 KiB into a ring of shared-memory entries - no tensor map per weight matrix.
//   h1 and h2 are needed again by the reverse layers (CELU' = 1 + min(h,0)/alpha).  They do not fit on the SM next to the
// weight ring (224 KiB per tile), so the forward epilogues also write them to the activation buffers in HBM and the reverse
// epilogues of the same CTA read them back a few microseconds later (L2 hits; 1.8 KB per atom and direction).
//
// TMEM (512 columns): region X = [0, 256) and region Y = [256, 448) hold the accumulators of alternate GEMMs of the chain
// (a GEMM with N > 128 is issued as two MMAs per K step, N = 128 at the region base and N - 128 at base + 128: both
// destinations stay 128-column aligned); Z = [448, 512) holds two A slots of 32 columns (hi 16 | lo 16).
//
// Chains (chosen per loaded system, nnp_fused_setup):
//   full   (active AEV columns kpad <= 192, e.g. water: 128):  F1 F2 F3 B3 B2 B1, input G (TMA), output dE/dG
//   middle (any kpad, e.g. 1024 for seven species):            F2 F3 B3 B2, input h1 (TMA), output delta1 in place;
//          F1 and B1 (K or N = kpad) run as launches of the unfused kernel before / after.
// Warp roles: 0 producer (TMA A tiles of the first GEMM + bulk weight copies), 1 MMA issue, 2-5 converters (first GEMM's
// A operand: fp32 tile in shared memory -> tf32 hi / lo slots), 6-13 epilogue (two warps per TMEM lane quarter, alternate
// 16-column chunks).
#include <cuda.h>

#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "nnp_internal.cuh"

namespace {

#include "tc_ptx.cuh"

constexpr int TILE_M = 128;
constexpr int KB = 32;                 // K block: fp32 elements of one 128-byte swizzle row
constexpr int CH = 16;                 // K chunk per A slot
constexpr int MAX_STAGES = 6;
constexpr int NW = 5;                  // weight ring entries
constexpr int W_ENTRY_BYTES = 32768;   // hi + lo tiles of up to 128 rows x 128 B
constexpr int NA = 2;                  // ring of first-GEMM A tiles
constexpr int A_TILE_BYTES = TILE_M * KB * 4;
constexpr int EPI_WARPS = 8;
constexpr int EPI_STG_LD = 20;
constexpr int EPI_STG_BYTES = 32 * EPI_STG_LD * 4;
constexpr int BAR_BYTES = 512;
constexpr int SMEM_BYTES = 1024 + NW * W_ENTRY_BYTES + NA * A_TILE_BYTES + BAR_BYTES + EPI_WARPS * EPI_STG_BYTES;
constexpr int THREADS = 14 * 32;
constexpr uint32_t COL_X = 0, COL_Y = 256, COL_Z = 448;
static_assert(SMEM_BYTES <= 227 * 1024, "shared memory budget");

enum FusedEpi {
    FE_FWD = 0,     // h = celu(acc + bias): stash h, hi/lo -> slots
    FE_OUT = 1,     // h3 = celu(acc + bias); e_atom += h3 . w4; delta3 = w4 celu'(h3): hi/lo -> slots
    FE_BWD = 2,     // delta = acc * celu'(stash): hi/lo -> slots
    FE_BWD_ST = 3,  // delta = acc * celu'(out): stored over out (last GEMM of the middle chain)
    FE_ST = 4,      // out = acc
    FE_RED = 5      // out += acc (vector reductions in memory: ensembles add into the same rows)
};

struct FusedStage {
    int K, N;            // K: columns of the A operand (multiple of 32); N: output columns (multiple of 32, <= 256 / 192)
    int epi;
    uint32_t w_off;      // byte offset of the packed weight tiles of this GEMM in the group's blob
    const float *bias;   // [N] (forward GEMMs)
    float *stash;        // rows of h: written by FE_FWD, read by FE_BWD (already offset to the group's first row)
    int ld_stash;
    int pad_;
};

struct alignas(64) FusedGroup {
    CUtensorMap mapA;    // A operand of the first GEMM: [M][K0] fp32, row pitch of the source buffer
    const uint8_t *wblob;
    const float *w4;
    float *e_atom;
    float *out;          // output rows of the last GEMM
    int ldo;
    int M, n_stages, tile0, n_tiles;
    int chunks_per_tile; // sum_j K_j / 16
    int y_first;         // accumulator region of GEMM j: (j & 1) ^ y_first ? Y : X
    int pad_;
    FusedStage st[MAX_STAGES];
};

__device__ __forceinline__ void bulk_load(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar)
                 : "memory");
}

__device__ __forceinline__ int find_group(const FusedGroup *__restrict__ groups, int n_groups, int t)
{
    int gi = 0;
    while (gi + 1 < n_groups && t >= groups[gi + 1].tile0) ++gi;
    return gi;
}

// rows of the two MMAs of a GEMM with N columns: 128 + (N - 128), or N alone
__device__ __forceinline__ int part_rows(int N, int p) { return p == 0 ? (N > 128 ? 128 : N) : N - 128; }

template <bool SPLIT3>
__global__ void __launch_bounds__(THREADS, 1)
k_mlp_fused(const FusedGroup *__restrict__ groups, int n_groups, const int *__restrict__ cta_tiles, float alpha)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t w_ring = smem_base, a_ring = smem_base + NW * W_ENTRY_BYTES;
    const uint32_t bar_base = a_ring + NA * A_TILE_BYTES;
    // barriers (8 B each)
    const uint32_t bar_wfull = bar_base, bar_wempty = bar_base + 8 * NW;
    const uint32_t bar_afull = bar_base + 16 * NW, bar_aempty = bar_afull + 8 * NA;
    const uint32_t bar_sready = bar_aempty + 8 * NA, bar_sfree = bar_sready + 16;
    const uint32_t bar_accf = bar_sfree + 16, bar_acce = bar_accf + 16;
    const uint32_t bar_tdone = bar_acce + 16; // every MMA of a tile has completed: both A slots are free for the next tile
    const uint32_t tmem_slot = bar_tdone + 8;
    const uint32_t stg_base = bar_base + BAR_BYTES;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int t_beg = cta_tiles[blockIdx.x], t_end = cta_tiles[blockIdx.x + 1];

    if (threadIdx.x == 0) {
        for (int e = 0; e < NW; ++e) { mbar_init(bar_wfull + 8 * e, 1); mbar_init(bar_wempty + 8 * e, 1); }
        for (int e = 0; e < NA; ++e) { mbar_init(bar_afull + 8 * e, 1); mbar_init(bar_aempty + 8 * e, 128); }
        for (int k = 0; k < 2; ++k) {
            mbar_init(bar_sready + 8 * k, 128);
            mbar_init(bar_sfree + 8 * k, 1);
            mbar_init(bar_accf + 8 * k, 1);
            mbar_init(bar_acce + 8 * k, EPI_WARPS * 32);
        }
        mbar_init(bar_tdone, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

    if (warp == 0) {
        // ===== producer: everything the MMA thread consumes from shared memory, in its order of use
        if (lane == 0) {
            uint32_t wi = 0, ai = 0;
            for (int t = t_beg; t < t_end; ++t) {
                const int gi = find_group(groups, n_groups, t);
                const FusedGroup &g = groups[gi];
                const int m0 = (t - g.tile0) * TILE_M;
                for (int j = 0; j < g.n_stages; ++j) {
                    const int K = g.st[j].K, N = g.st[j].N;
                    const int parts = N > 128 ? 2 : 1;
                    const uint8_t *wsrc = g.wblob + g.st[j].w_off;
                    for (int kb = 0; kb < K / KB; ++kb) {
                        if (j == 0) {
                            const uint32_t e = ai % NA;
                            mbar_wait(bar_aempty + 8 * e, ((ai / NA) & 1) ^ 1, 150, (t - t_beg) * 100 + kb);
                            mbar_expect_tx(bar_afull + 8 * e, A_TILE_BYTES);
                            tma_load_2d(a_ring + e * A_TILE_BYTES, &g.mapA, kb * KB, m0, bar_afull + 8 * e);
                            ++ai;
                        }
                        for (int p = 0; p < parts; ++p, ++wi) {
                            const uint32_t e = wi % NW;
                            const uint32_t rows = (uint32_t)part_rows(N, p);
                            const uint32_t bytes = (SPLIT3 ? 2u : 1u) * rows * 128u; // hi tile first, lo tile behind it
                            mbar_wait(bar_wempty + 8 * e, ((wi / NW) & 1) ^ 1, 100 + j, (t - t_beg) * 100 + kb);
                            mbar_expect_tx(bar_wfull + 8 * e, bytes);
                            bulk_load(w_ring + e * W_ENTRY_BYTES, wsrc, bytes, bar_wfull + 8 * e);
                            wsrc += 2u * rows * 128u;
                        }
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issue (whole warp walks the loop, one elected lane issues)
        uint32_t wi = 0, ci = 0, useX = 0, useY = 0;
        for (int t = t_beg; t < t_end; ++t) {
            const int gi = find_group(groups, n_groups, t);
            const FusedGroup &g = groups[gi];
            for (int j = 0; j < g.n_stages; ++j) {
                const int K = g.st[j].K, N = g.st[j].N;
                const int parts = N > 128 ? 2 : 1;
                // regions alternate; the chain starts in the one that puts its widest GEMMs (N <= 256) into X
                const int in_y = (j & 1) ^ g.y_first;
                const uint32_t acc = tmem_base + (in_y ? COL_Y : COL_X);
                uint32_t &use = in_y ? useY : useX;
                mbar_wait(bar_acce + 8 * in_y, (use & 1) ^ 1, 200 + j, t - t_beg); // the epilogue has drained the previous accumulator of this region
                tc_fence_after();
                const uint32_t idesc0 = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(part_rows(N, 0) >> 3) << 17) | ((uint32_t)(TILE_M >> 4) << 24);
                const uint32_t idesc1 = parts > 1 ? (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(part_rows(N, 1) >> 3) << 17) | ((uint32_t)(TILE_M >> 4) << 24) : 0u;
                for (int kb = 0; kb < K / KB; ++kb) {
                    const uint32_t e0 = wi % NW, e1 = (wi + 1) % NW;
                    mbar_wait(bar_wfull + 8 * e0, (wi / NW) & 1, 220 + j, (t - t_beg) * 100 + kb);
                    if (parts > 1) mbar_wait(bar_wfull + 8 * e1, ((wi + 1) / NW) & 1, 230 + j, (t - t_beg) * 100 + kb);
                    const uint32_t b0 = w_ring + e0 * W_ENTRY_BYTES, b1 = w_ring + e1 * W_ENTRY_BYTES;
                    const uint64_t d0hi = make_kmajor_sw128_desc(b0), d0lo = make_kmajor_sw128_desc(b0 + (uint32_t)part_rows(N, 0) * 128u);
                    const uint64_t d1hi = make_kmajor_sw128_desc(b1), d1lo = make_kmajor_sw128_desc(b1 + (uint32_t)(parts > 1 ? part_rows(N, 1) : 8) * 128u);
#pragma unroll
                    for (int h = 0; h < 2; ++h, ++ci) {
                        const uint32_t k = ci & 1;
                        mbar_wait(bar_sready + 8 * k, (ci >> 1) & 1, 240 + j, (t - t_beg) * 100 + 2 * kb + h);
                        tc_fence_after();
                        const uint32_t a_hi = tmem_base + COL_Z + 32u * k, a_lo = a_hi + 16;
                        if (elect_one()) {
#pragma unroll
                            for (int ks = 0; ks < 2; ++ks) {
                                const uint64_t koff = (uint64_t)(((2 * h + ks) * 8 * 4) >> 4);
                                const uint32_t first = (kb | h | ks) ? 1u : 0u;
                                if (SPLIT3) {
                                    mma_tf32_ts(acc, a_lo + 8 * ks, d0hi + koff, idesc0, first);
                                    mma_tf32_ts(acc, a_hi + 8 * ks, d0lo + koff, idesc0, 1u);
                                    mma_tf32_ts(acc, a_hi + 8 * ks, d0hi + koff, idesc0, 1u);
                                    if (parts > 1) {
                                        mma_tf32_ts(acc + 128, a_lo + 8 * ks, d1hi + koff, idesc1, first);
                                        mma_tf32_ts(acc + 128, a_hi + 8 * ks, d1lo + koff, idesc1, 1u);
                                        mma_tf32_ts(acc + 128, a_hi + 8 * ks, d1hi + koff, idesc1, 1u);
                                    }
                                } else {
                                    mma_tf32_ts(acc, a_hi + 8 * ks, d0hi + koff, idesc0, first);
                                    if (parts > 1) mma_tf32_ts(acc + 128, a_hi + 8 * ks, d1hi + koff, idesc1, first);
                                }
                            }
                            tc_commit(bar_sfree + 8 * k);
                            if (h == 1) {
                                tc_commit(bar_wempty + 8 * e0);
                                if (parts > 1) tc_commit(bar_wempty + 8 * e1);
                                if (kb + 1 == K / KB) {
                                    tc_commit(bar_accf + 8 * in_y);
                                    if (j + 1 == g.n_stages) tc_commit(bar_tdone);
                                }
                            }
                        }
                        __syncwarp();
                    }
                    wi += parts;
                }
                ++use;
            }
        }
    } else if (warp < 6) {
        // ===== converters: A operand of the first GEMM (fp32 rows from HBM through the TMA ring) -> hi / lo slots
        const int quarter = warp & 3;
        const int row = quarter * 32 + lane;
        const uint32_t lane_addr = tmem_base + ((uint32_t)(quarter * 32) << 16);
        uint32_t ai = 0, ci = 0;
        for (int t = t_beg; t < t_end; ++t) {
            const int gi = find_group(groups, n_groups, t);
            const FusedGroup &g = groups[gi];
            const int nkb = g.st[0].K / KB;
            // The slot barriers count in parities: a converter that ran a whole tile ahead would take the completion of
            // ANY earlier use of a slot for the one it waits for.  The epilogue warps are held back by the accumulator
            // barriers; the converters wait here until the previous tile has consumed its last chunk.
            if (t > t_beg) mbar_wait(bar_tdone, (uint32_t)(t - t_beg - 1) & 1, 320, t - t_beg);
            for (int kb = 0; kb < nkb; ++kb, ++ai) {
                const uint32_t e = ai % NA;
                mbar_wait(bar_afull + 8 * e, (ai / NA) & 1, 300, (t - t_beg) * 100 + kb);
                const uint32_t arow = a_ring + e * A_TILE_BYTES + row * 128;
                float x[32];
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    const uint32_t addr = arow + (uint32_t)((c ^ (row & 7)) << 4);
                    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(x[4 * c]), "=f"(x[4 * c + 1]), "=f"(x[4 * c + 2]), "=f"(x[4 * c + 3]) : "r"(addr));
                }
                mbar_arrive(bar_aempty + 8 * e); // the tile is in registers
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const uint32_t c = ci + 2 * kb + h, k = c & 1;
                    uint32_t v[32];
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        const float xv = x[16 * h + q];
                        const uint32_t hi = tf32_round(xv);
                        v[q] = hi;
                        v[16 + q] = SPLIT3 ? tf32_round(xv - __uint_as_float(hi)) : 0u;
                    }
                    mbar_wait(bar_sfree + 8 * k, ((c >> 1) & 1) ^ 1, 310, (t - t_beg) * 100 + 2 * kb + h);
                    tc_fence_after();
                    tmem_st32(lane_addr + COL_Z + 32u * k, v);
                    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                    tc_fence_before();
                    mbar_arrive(bar_sready + 8 * k);
                }
            }
            ci += (uint32_t)g.chunks_per_tile;
        }
    } else {
        // ===== epilogue: warps 6..13 -> TMEM lane quarters 2,3,0,1,2,3,0,1; set 0 (warps 6-9) takes the even 16-column
        // chunks of an accumulator, set 1 the odd ones.  This thread owns accumulator row `row`.
        const int ew = warp - 6;
        const int quarter = warp & 3;
        const int set = ew >> 2;
        const int row = quarter * 32 + lane;
        const uint32_t lane_addr = tmem_base + ((uint32_t)(quarter * 32) << 16);
        const uint32_t stg = stg_base + (uint32_t)ew * EPI_STG_BYTES;
        const uint32_t my_row = stg + (uint32_t)lane * (EPI_STG_LD * 4);
        const int sub_r = (lane >> 3) + 4 * ((lane >> 2) & 1), sub_c = (lane & 3) * 4;
        const float inv_alpha = 1.0f / alpha;
        uint32_t ci = 0, useX = 0, useY = 0;
        for (int t = t_beg; t < t_end; ++t) {
            const int gi = find_group(groups, n_groups, t);
            const FusedGroup &g = groups[gi];
            const int m0 = (t - g.tile0) * TILE_M;
            const int mrow0 = m0 + quarter * 32;
            const int m = mrow0 + lane;
            const bool rowok = m < g.M;
            uint32_t cj = ci + (uint32_t)(g.st[0].K / CH); // chunk index of the first slot this stage's epilogue produces
            for (int j = 0; j < g.n_stages; ++j) {
                const int N = g.st[j].N, epi = g.st[j].epi;
                const int in_y = (j & 1) ^ g.y_first;
                const uint32_t acc_col = in_y ? COL_Y : COL_X;
                uint32_t &use = in_y ? useY : useX;
                const bool fwd = epi == FE_FWD || epi == FE_OUT;
                const bool rd_prev = epi == FE_BWD || epi == FE_BWD_ST;   // reads rows of h for CELU'
                const bool to_slot = epi == FE_FWD || epi == FE_OUT || epi == FE_BWD;
                const bool wr_rows = epi == FE_FWD || epi == FE_BWD_ST || epi == FE_ST || epi == FE_RED;
                // rows read (h for CELU') and rows written (h stash, or the chain's output)
                const float *rd_base = epi == FE_BWD ? g.st[j].stash : g.out;
                const int rd_ld = epi == FE_BWD ? g.st[j].ld_stash : g.ldo;
                float *wr_base = epi == FE_FWD ? g.st[j].stash : g.out;
                const int wr_ld = epi == FE_FWD ? g.st[j].ld_stash : g.ldo;
                const float *bias = g.st[j].bias, *w4 = g.w4;
                float esum = 0.f;
                float bias_l = 0.f, w4_l = 0.f;
                float4 pre[4];
                auto prefetch = [&](int c0) {
                    if (fwd) bias_l = lane < CH ? bias[c0 + lane] : 0.f;
                    if (epi == FE_OUT) w4_l = lane < CH ? w4[c0 + lane] : 0.f;
                    if (rd_prev) {
                        const float *cb = rd_base + (size_t)mrow0 * rd_ld + c0;
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const int r = i * 8 + sub_r;
                            pre[i] = mrow0 + r < g.M ? *reinterpret_cast<const float4 *>(cb + (size_t)r * rd_ld + sub_c)
                                                     : make_float4(0.f, 0.f, 0.f, 0.f);
                        }
                    }
                };
                const int c_first = set * CH;
                if (c_first < N) prefetch(c_first);
                mbar_wait(bar_accf + 8 * in_y, use & 1, 400 + j, t - t_beg);
                tc_fence_after();
                for (int c0 = c_first; c0 < N; c0 += 2 * CH) {
                    const float bias_c = bias_l, w4_c = w4_l;
                    if (rd_prev) {
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const int r = i * 8 + sub_r;
                            asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(stg + (uint32_t)(r * EPI_STG_LD + sub_c) * 4), "f"(pre[i].x), "f"(pre[i].y), "f"(pre[i].z), "f"(pre[i].w) : "memory");
                        }
                        __syncwarp();
                    }
                    if (c0 + 2 * CH < N) prefetch(c0 + 2 * CH);
                    uint32_t a[16];
                    tmem_ld16(lane_addr + acc_col + (uint32_t)c0, a);
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    uint32_t sl[32];
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        float4 prev = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (rd_prev)
                            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(prev.x), "=f"(prev.y), "=f"(prev.z), "=f"(prev.w) : "r"(my_row + q * 16));
                        const float pv[4] = {prev.x, prev.y, prev.z, prev.w};
                        float ov[4], hv[4];
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            float v = __uint_as_float(a[4 * q + e]);
                            float bv = 0.f, wv = 0.f;
                            bv = __shfl_sync(0xffffffffu, bias_c, 4 * q + e);
                            wv = __shfl_sync(0xffffffffu, w4_c, 4 * q + e);
                            hv[e] = 0.f;
                            if (epi == FE_FWD) { v = celu_fwd(v + bv, alpha, inv_alpha); hv[e] = v; }
                            else if (epi == FE_OUT) {
                                const float hh = celu_fwd(v + bv, alpha, inv_alpha);
                                esum = fmaf(hh, wv, esum);
                                v = wv * celu_grad_from_h(hh, inv_alpha);
                            } else if (rd_prev) v *= celu_grad_from_h(pv[e], inv_alpha);
                            ov[e] = v;
                            const uint32_t hi = tf32_round(v);
                            sl[4 * q + e] = hi;
                            sl[16 + 4 * q + e] = SPLIT3 ? tf32_round(v - __uint_as_float(hi)) : 0u;
                        }
                        if (wr_rows) {
                            if (rd_prev) __syncwarp(); // (same thread re-uses its own staged row: no hazard across lanes here)
                            asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(my_row + q * 16), "f"(epi == FE_FWD ? hv[0] : ov[0]), "f"(epi == FE_FWD ? hv[1] : ov[1]), "f"(epi == FE_FWD ? hv[2] : ov[2]), "f"(epi == FE_FWD ? hv[3] : ov[3]) : "memory");
                        }
                    }
                    if (to_slot) {
                        const uint32_t c = cj + (uint32_t)(c0 / CH), k = c & 1;
                        mbar_wait(bar_sfree + 8 * k, ((c >> 1) & 1) ^ 1, 420 + j, (t - t_beg) * 1000 + c0);
                        tc_fence_after();
                        tmem_st32(lane_addr + COL_Z + 32u * k, sl);
                        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                        tc_fence_before();
                        mbar_arrive(bar_sready + 8 * k);
                    }
                    if (wr_rows) {
                        __syncwarp();
                        float *cbase = wr_base + (size_t)mrow0 * wr_ld + c0;
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const int r = i * 8 + sub_r;
                            if (mrow0 + r < g.M) {
                                float4 v;
                                asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(stg + (uint32_t)(r * EPI_STG_LD + sub_c) * 4));
                                if (epi == FE_RED) atomicAdd(reinterpret_cast<float4 *>(cbase + (size_t)r * wr_ld + sub_c), v);
                                else *reinterpret_cast<float4 *>(cbase + (size_t)r * wr_ld + sub_c) = v;
                            }
                        }
                        __syncwarp();
                    } else if (rd_prev) {
                        __syncwarp(); // every lane has read its staged row before the next chunk overwrites the staging
                    }
                }
                tc_fence_before();
                mbar_arrive(bar_acce + 8 * in_y);
                ++use;
                if (epi == FE_OUT && rowok) atomicAdd(g.e_atom + m, esum);
                if (to_slot) cj += (uint32_t)(N / CH);
            }
            ci = cj;
        }
    }
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
    }
}

// Packs one weight matrix Bt [N][K] (K contiguous; the B operand of D = A . Bt^T) into the tile images the kernel copies
// with one bulk load each: for every K block of 32 and part p (rows [0,128) / [128,N)): the tf32-hi tile then the tf32-lo
// tile, rows of 128 B, 16-byte chunk c of row r stored at chunk position c ^ (r & 7) (128-byte swizzle).
__global__ void k_pack_weights(const float *__restrict__ Bt, int N, int K, int ldb, uint8_t *__restrict__ dst)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x; // one 16-byte chunk of one row of one K block
    const int nkb = K / KB;
    if (idx >= N * nkb * 8) return;
    const int c = idx & 7, n = (idx >> 3) % N, kb = (idx >> 3) / N;
    const int p = n >= 128 ? 1 : 0, rows = p == 0 ? (N > 128 ? 128 : N) : N - 128, r = n - 128 * p;
    // K block kb: [part 0: hi rows0 x 128 | lo rows0 x 128][part 1: hi | lo]
    const size_t kb_bytes = (size_t)2 * N * 128;
    uint8_t *tile = dst + kb * kb_bytes + (p ? (size_t)2 * (N > 128 ? 128 : N) * 128 : 0);
    const float4 v = *reinterpret_cast<const float4 *>(Bt + (size_t)n * ldb + kb * KB + 4 * c);
    const float x[4] = {v.x, v.y, v.z, v.w};
    uint32_t hi[4], lo[4];
    for (int e = 0; e < 4; ++e) {
        hi[e] = (__float_as_uint(x[e]) + 0x1000u) & 0xffffe000u;
        lo[e] = (__float_as_uint(x[e] - __uint_as_float(hi[e])) + 0x1000u) & 0xffffe000u;
    }
    const size_t off = (size_t)r * 128 + (size_t)((c ^ (r & 7)) << 4);
    *reinterpret_cast<uint4 *>(tile + off) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4 *>(tile + (size_t)rows * 128 + off) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;

bool load_encode()
{
    if (g_encode) return true;
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) return false;
    g_encode = (EncodeTiledFn)fn;
    return true;
}

bool make_map_a(CUtensorMap *m, const float *base, int rows, int cols, int ld)
{
    cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)ld * 4};
    cuuint32_t box[2] = {(cuuint32_t)KB, (cuuint32_t)TILE_M};
    cuuint32_t estr[2] = {1, 1};
    return g_encode(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void *)base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

} // namespace

struct nnp_fused {
    int kind;                    // 0: not usable for the loaded system, 1: full chain, 2: middle chain
    int n_groups, n_tiles, grid;
    FusedGroup *d_groups;        // [n_nets * S]
    int *d_cta_tiles;            // [grid + 1]
    uint8_t *d_wblob;            // packed weights of every (network, species): sized at first use for the full layout
    size_t wblob_bytes;
    size_t w_off[64][MAX_STAGES + 1]; // per (network, species): byte offsets of F1 F2 F3 B3 B2 B1 in the blob
    unsigned packed_mask;        // species mask the layer-1 tiles were packed for (0: nothing packed yet)
    int num_sms;
};

void nnp_fused_destroy(nnp_ctx *c)
{
    nnp_fused *f = c->fused;
    if (!f) return;
    void (*fr)(nnp_ctx *, void *) = [](nnp_ctx *cc, void *p) {
        if (!p) return;
        if (cc->dealloc_fn) cc->dealloc_fn(p, cc->alloc_user); else cudaFree(p);
    };
    fr(c, f->d_groups); fr(c, f->d_cta_tiles); fr(c, f->d_wblob);
    delete f;
    c->fused = nullptr;
}

static void *fused_alloc(nnp_ctx *c, size_t bytes)
{
    if (c->alloc_fn) return c->alloc_fn(bytes ? bytes : 256, c->alloc_user);
    void *p = nullptr;
    if (cudaMalloc(&p, bytes ? bytes : 256) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return p;
}

// Decides whether (and which chain of) the fused kernel serves the loaded system, packs the weights (once per species
// set: the layer-1 tiles depend on the active AEV columns) and builds the group table and the per-CTA tile ranges.
// Called by nnp_set_system after the layout is known.  Returns NNP_OK also when the fused path is not applicable
// (c->fused->kind = 0: the six-launch path runs).
int nnp_fused_setup(nnp_ctx *c)
{
    if (!c->tc_mode || c->no_fused) return NNP_OK;
    if (!load_encode()) { c->err = "cuTensorMapEncodeTiled entry point not available"; return NNP_ECUDA; }
    const int S = c->S, nn = c->n_nets;
    if (nn * S > 64) return NNP_OK;
    if (!c->fused) {
        c->fused = new nnp_fused();
        memset(c->fused, 0, sizeof(nnp_fused));
        cudaDeviceGetAttribute(&c->fused->num_sms, cudaDevAttrMultiProcessorCount, c->device);
        if (c->fused->num_sms <= 0) c->fused->num_sms = 148;
    }
    nnp_fused *f = c->fused;
    f->kind = 0;
    const int kpad = c->aev.kpad;
    // widths the TMEM layout can hold: X (256 columns): h1, h3; Y (192): h2 and, in the full chain, kpad
    for (int s = 0; s < S; ++s)
        if (c->widths[s][1] > 256 || c->widths[s][2] > 192 || c->widths[s][3] > 256) return NNP_OK;
    const int kind = kpad <= 192 ? 1 : 2;
    // ---- packed weights: per (net, species) the six matrices in chain order; sized for the largest layout once
    if (!f->d_wblob) {
        size_t tot = 0;
        for (int net = 0; net < nn; ++net)
            for (int s = 0; s < S; ++s) {
                const size_t k0 = c->kpad_full < 192 ? c->kpad_full : 192, h1 = c->widths[s][1], h2 = c->widths[s][2], h3 = c->widths[s][3];
                tot += 8 * (2 * k0 * h1 + 2 * h1 * h2 + 2 * h2 * h3);
            }
        f->d_wblob = (uint8_t *)fused_alloc(c, tot);
        if (!f->d_wblob) { c->err = "fused MLP: weight tile allocation failed"; return NNP_ENOMEM; }
        f->wblob_bytes = tot;
        f->d_groups = (FusedGroup *)fused_alloc(c, sizeof(FusedGroup) * 64);
        f->d_cta_tiles = (int *)fused_alloc(c, sizeof(int) * (f->num_sms + 1));
        if (!f->d_groups || !f->d_cta_tiles) { c->err = "fused MLP: table allocation failed"; return NNP_ENOMEM; }
        f->packed_mask = 0;
    }
    auto pack = [&](const float *Bt, int N, int K, int ldb, uint8_t *dst) {
        const int total = N * (K / KB) * 8;
        k_pack_weights<<<nnp_div_up(total, 256), 256, 0, c->stream>>>(Bt, N, K, ldb, dst);
        c->launches += 1;
    };
    const bool repack_l1 = f->packed_mask != c->present_mask;
    const bool first_pack = f->packed_mask == 0;
    {
        size_t o = 0;
        for (int net = 0; net < nn; ++net)
            for (int s = 0; s < S; ++s) {
                const int q = net * S + s;
                const int h1 = c->widths[s][1], h2 = c->widths[s][2], h3 = c->widths[s][3];
                const LayerW *L = &c->layers[((size_t)net * S + s) * NNP_NLAYERS];
                const Layer1C &l1 = c->l1c[(size_t)net * S + s];
                const size_t k0 = c->kpad_full < 192 ? c->kpad_full : 192; // layer-1 tiles exist for the full chain only
                // F1: B = W1^T [h1][kpad]; F2: W2^T [h2][h1]; F3: W3^T [h3][h2]; B3: W3 [h2][h3]; B2: W2 [h1][h2]; B1: W1 [kpad][h1]
                f->w_off[q][0] = o; o += 8 * k0 * h1;
                f->w_off[q][1] = o; o += 8 * (size_t)h1 * h2;
                f->w_off[q][2] = o; o += 8 * (size_t)h2 * h3;
                f->w_off[q][3] = o; o += 8 * (size_t)h2 * h3;
                f->w_off[q][4] = o; o += 8 * (size_t)h1 * h2;
                f->w_off[q][5] = o; o += 8 * k0 * h1;
                f->w_off[q][6] = o;
                if (first_pack) {
                    pack(L[1].Wt, h2, h1, h1, f->d_wblob + f->w_off[q][1]);
                    pack(L[2].Wt, h3, h2, h2, f->d_wblob + f->w_off[q][2]);
                    pack(L[2].W, h2, h3, h3, f->d_wblob + f->w_off[q][3]);
                    pack(L[1].W, h1, h2, h2, f->d_wblob + f->w_off[q][4]);
                }
                if (repack_l1 && kind == 1) {
                    pack(l1.Wt, h1, kpad, kpad, f->d_wblob + f->w_off[q][0]);
                    pack(l1.W, kpad, h1, h1, f->d_wblob + f->w_off[q][5]);
                }
            }
    }
    if (kind == 1) f->packed_mask = c->present_mask;
    else if (first_pack) f->packed_mask = 0x80000000u; // middle GEMMs packed, no layer-1 tiles

    // ---- groups (one per network and species present) and tiles
    std::vector<FusedGroup> groups;
    std::vector<long long> cost;
    int tiles = 0;
    for (int net = 0; net < nn; ++net)
        for (int s = 0; s < S; ++s) {
            const int off = c->bucket_off[s], M = c->bucket_off[s + 1] - off;
            if (M == 0) continue;
            const int q = net * S + s;
            const int h1 = c->widths[s][1], h2 = c->widths[s][2], h3 = c->widths[s][3];
            const LayerW *L = &c->layers[((size_t)net * S + s) * NNP_NLAYERS];
            float *H0 = c->H[0] + ((size_t)net * c->max_atoms + off) * c->hmax[0];
            float *H1 = c->H[1] + ((size_t)net * c->max_atoms + off) * c->hmax[1];
            FusedGroup g;
            memset(&g, 0, sizeof(g));
            g.wblob = f->d_wblob;
            g.w4 = L[3].W;
            g.e_atom = c->e_atom + off;
            g.M = M;
            g.tile0 = tiles;
            g.n_tiles = nnp_div_up(M, TILE_M);
            auto stage = [&](int j, int K, int N, int epi, size_t w_off, const float *bias, float *stash, int ld) {
                FusedStage &st = g.st[j];
                st.K = K; st.N = N; st.epi = epi; st.w_off = (uint32_t)w_off; st.bias = bias; st.stash = stash; st.ld_stash = ld;
            };
            if (f->w_off[q][6] > 0xffffffffull) { c->err = "fused MLP: weight blob exceeds 4 GiB"; return NNP_EINVAL; }
            if (kind == 1) {
                g.n_stages = 6;
                if (!make_map_a(&g.mapA, c->G + (size_t)off * kpad, M, kpad, kpad)) { c->err = "cuTensorMapEncodeTiled failed"; return NNP_ECUDA; }
                stage(0, kpad, h1, FE_FWD, f->w_off[q][0], L[0].b, H0, c->hmax[0]);
                stage(1, h1, h2, FE_FWD, f->w_off[q][1], L[1].b, H1, c->hmax[1]);
                stage(2, h2, h3, FE_OUT, f->w_off[q][2], L[2].b, nullptr, 0);
                stage(3, h3, h2, FE_BWD, f->w_off[q][3], nullptr, H1, c->hmax[1]);
                stage(4, h2, h1, FE_BWD, f->w_off[q][4], nullptr, H0, c->hmax[0]);
                stage(5, h1, kpad, nn > 1 ? FE_RED : FE_ST, f->w_off[q][5], nullptr, nullptr, 0);
                g.out = c->dG + (size_t)off * kpad;
                g.ldo = kpad;
                g.y_first = 0; // F1 X, F2 Y, F3 X, B3 Y, B2 X, B1 Y (kpad <= 192)
            } else {
                g.n_stages = 4;
                g.y_first = 1; // F2 Y, F3 X, B3 Y, B2 X (h1 <= 256)
                if (!make_map_a(&g.mapA, H0, M, h1, c->hmax[0])) { c->err = "cuTensorMapEncodeTiled failed"; return NNP_ECUDA; }
                stage(0, h1, h2, FE_FWD, f->w_off[q][1], L[1].b, H1, c->hmax[1]);
                stage(1, h2, h3, FE_OUT, f->w_off[q][2], L[2].b, nullptr, 0);
                stage(2, h3, h2, FE_BWD, f->w_off[q][3], nullptr, H1, c->hmax[1]);
                stage(3, h2, h1, FE_BWD_ST, f->w_off[q][4], nullptr, nullptr, 0);
                g.out = H0;
                g.ldo = c->hmax[0];
            }
            long long cst = 0;
            for (int j = 0; j < g.n_stages; ++j) {
                g.chunks_per_tile += g.st[j].K / CH;
                cst += (long long)(g.st[j].K / 8) * 3 * (g.st[j].N / 2) + 1500; // MMA cycles + the hand-over bubble of a GEMM
            }
            tiles += g.n_tiles;
            groups.push_back(g);
            cost.push_back(cst);
        }
    f->n_groups = (int)groups.size();
    f->n_tiles = tiles;
    if (tiles == 0) return NNP_OK;
    // contiguous tile ranges of equal cost
    int grid = tiles < f->num_sms ? tiles : f->num_sms;
    const char *dbg = getenv("NNP_FUSED_DEBUG");
    if (dbg && dbg[0] == '2') grid = (tiles + 1) / 2;
    std::vector<int> cta(grid + 1, tiles);
    {
        long long total = 0;
        for (size_t q = 0; q < groups.size(); ++q) total += cost[q] * groups[q].n_tiles;
        cta[0] = 0;
        long long acc = 0;
        int b = 1;
        for (size_t q = 0; q < groups.size() && b < grid; ++q)
            for (int k = 0; k < groups[q].n_tiles && b < grid; ++k) {
                acc += cost[q];
                while (b < grid && acc * grid >= total * b) { cta[b] = groups[q].tile0 + k + 1; ++b; }
            }
        cta[grid] = tiles;
        for (int k = 1; k <= grid; ++k)
            if (cta[k] < cta[k - 1]) cta[k] = cta[k - 1];
    }
    if (dbg && (dbg[0] == '1' || dbg[0] == '2'))
        for (int k = 0; k <= grid; ++k) cta[k] = (int)((long long)tiles * k / grid);
    f->grid = grid;
    if (cudaMemcpyAsync(f->d_groups, groups.data(), sizeof(FusedGroup) * groups.size(), cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaMemcpyAsync(f->d_cta_tiles, cta.data(), sizeof(int) * (grid + 1), cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess) { // the host vectors go out of scope
        c->err = std::string("fused MLP: table upload failed: ") + cudaGetErrorString(cudaGetLastError());
        return NNP_ECUDA;
    }
    f->kind = kind;
    return NNP_OK;
}

int nnp_fused_kind(const nnp_ctx *c) { return c->fused ? c->fused->kind : 0; }

// Enqueues the fused chain.  kind 1: replaces all six GEMM launches; kind 2: replaces the four middle ones.
void nnp_launch_mlp_fused(nnp_ctx *c)
{
    nnp_fused *f = c->fused;
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(k_mlp_fused<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        cudaFuncSetAttribute(k_mlp_fused<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        attr_set = true;
    }
    if (c->mm_mode == NNP_MM_3XTF32_TC)
        k_mlp_fused<true><<<f->grid, THREADS, SMEM_BYTES, c->stream>>>(f->d_groups, f->n_groups, f->d_cta_tiles, c->alpha);
    else
        k_mlp_fused<false><<<f->grid, THREADS, SMEM_BYTES, c->stream>>>(f->d_groups, f->n_groups, f->d_cta_tiles, c->alpha);
    c->launches += 1;
}
