// Stage 3/4, mm_mode = NNP_MM_3XTF32_TC / NNP_MM_TF32_TC: species-grouped GEMMs on the 5th-generation tensor
// cores (tcgen05.mma kind::tf32, accumulators in TMEM, operands by TMA) with the layer epilogues fused.
// ChemicalNet.  Precision (only full fp32 matmuls conserve energy; TF32 does
// not): the default mode is 3xTF32 -- every fp32 operand x is split into hi = tf32(x) and lo = tf32(x - hi), and
// A.B is accumulated in fp32 as A_lo.B_hi + A_hi.B_lo + A_hi.B_hi, which carries ~21 mantissa bits per operand.
// Weights are split once at nnp_create; activations are split on the fly inside the kernel.
//
// One CTA computes one 128-row (atoms) x N (<= 256 features) output tile:
//   warp 0   TMA producer: per 32-wide K block, the fp32 A tile [128][32] and the B_hi / B_lo tiles [N][32]
//            (K-major, 128-byte swizzle) into a 2-stage shared-memory ring, mbarrier complete_tx.
//   warps 2-5 converters: each thread owns one A row: reads it from the swizzled tile (conflict-free LDS.128),
//            splits it into tf32 hi / lo and writes both into TMEM (tcgen05.st) -- A is fed to the tensor core
//            from TMEM (".ts" form), so shared-memory bandwidth is spent on B only.
//   warp 1   one elected thread issues tcgen05.mma (3 per 8-wide K step in 3xTF32 mode); tcgen05.commit
//            releases the stage (shared memory + TMEM A slot) and finally signals the accumulator.
//   warps 2-5 epilogue: tcgen05.ld the accumulator row, apply bias/CELU/CELU'/output-layer dot, store.
#include <cuda.h>

#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "nnp_internal.cuh"

namespace {

constexpr int TILE_M = 128;
constexpr int BLOCK_K = 32;               // fp32 elements = one 128-byte swizzle row
constexpr int UMMA_K = 8;                 // tf32
constexpr int NT_MAX = 192;               // columns per output tile = the layer width up to 192; wider layers in equal parts
constexpr int STAGES_MAX = 4;             // shared-memory ring: 4 stages of 48 KiB (NT <= 128) or 3 of up to 64 KiB
constexpr int A_TILE_BYTES = TILE_M * BLOCK_K * 4;          // 16 KiB
constexpr int EPI_WARPS = 8;                                     // two per TMEM lane quarter, on alternate column chunks
constexpr int EPI_CW = 16;                                       // columns per epilogue chunk
constexpr int EPI_STG_LD = 20;                                   // floats per staged row (16-byte aligned, conflict-free)
constexpr int EPI_STG_BYTES = 32 * EPI_STG_LD * 4;               // per epilogue warp: one 32 x 16 chunk
constexpr int SMEM_FIXED = 1024 /*align*/ + 256 /*barriers*/ + EPI_WARPS * EPI_STG_BYTES;
constexpr int SMEM_LIMIT = 227 * 1024;
constexpr int TMEM_COLS = 512;
// TMEM: two accumulator buffers at columns 0 and acc_stride (128 / 160 / 192), behind them a_slots = 4 / 3 / 2 A slots
// (hi 32 + lo 32 columns); K block `it` uses slot it % a_slots and shared-memory stage it % stages (a_slots <= stages).
constexpr int THREADS = 576;              // warp 0 TMA, warp 1 MMA, warps 2-9 converters (two groups), warps 10-17 epilogue

struct TcGroup {
    CUtensorMap mapA, mapBhi, mapBlo;
    float *C;
    const float *bias, *w4;
    float *e_atom;
    int M, N, K, ldc;
    int NT;        // columns per tile
    int n_tiles_n; // N / NT
};

struct TcBatch {
    TcGroup g[NNP_MAX_GROUPS];
    int n_groups;
    int tile_off[NNP_MAX_GROUPS + 1]; // prefix sum of (m tiles x n tiles) per group
    int n_tiles;
    int tile_cost[NNP_MAX_GROUPS]; // bytes moved per tile of the group, in units of 128 B
    long long cost_total;
    int stages, stage_bytes, b_tile_bytes; // ring depth; 16 KiB + 2 * b_tile_bytes; nt_max * 128
    int acc_stride, a_slots;
    float alpha;
};


#include "tc_ptx.cuh"

// tile index -> (group, m0, n0)
struct TileCoord { int gi, m0, n0; };
__device__ __forceinline__ TileCoord tile_coord(const TcBatch &batch, int t)
{
    int gi = 0;
    while (gi + 1 < batch.n_groups && t >= batch.tile_off[gi + 1]) ++gi;
    const int r = t - batch.tile_off[gi];
    const int ntn = batch.g[gi].n_tiles_n;
    const int mt = r / ntn, nt = r - mt * ntn;
    return TileCoord{gi, mt * TILE_M, nt * batch.g[gi].NT};
}

// first tile whose cumulative cost reaches x
__device__ __forceinline__ int tile_at_cost(const TcBatch &batch, long long x)
{
    for (int gi = 0; gi < batch.n_groups; ++gi) {
        const long long w = batch.tile_cost[gi], n = batch.tile_off[gi + 1] - batch.tile_off[gi];
        if (x < w * n) return batch.tile_off[gi] + (int)((x + w - 1) / w);
        x -= w * n;
    }
    return batch.n_tiles;
}

// Persistent: CTA c processes the contiguous tile range [c T / G, (c+1) T / G); the two n-halves of an m-tile are
// adjacent, so the second read of the A tile hits L2.  The smem/TMEM-A ring (4 stages) and the two accumulator
// buffers run across tile boundaries: the epilogue of tile i overlaps the conversion + MMAs of tile i+1.
template <int EPI, bool SPLIT3>
__global__ void __launch_bounds__(THREADS, 1)
k_gemm_tc(const __grid_constant__ TcBatch batch)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const int S = batch.stages, T = batch.a_slots;
    const uint32_t stage_bytes = (uint32_t)batch.stage_bytes, blo_off = A_TILE_BYTES + (uint32_t)batch.b_tile_bytes;
    const uint32_t a_col0 = 2u * (uint32_t)batch.acc_stride;
    const uint32_t bar_base = smem_base + S * stage_bytes;
    // barriers (8 B each): full[4] @0, aready[4] @32, empty[4] @64, acc_full[2] @96, acc_empty[2] @112; tmem ptr @128
    const uint32_t bar_full = bar_base, bar_aready = bar_base + 32, bar_empty = bar_base + 64;
    const uint32_t bar_accf = bar_base + 96, bar_acce = bar_base + 112;
    const uint32_t tmem_slot = bar_base + 128;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // contiguous tile ranges of equal COST, not equal count: a hydrogen tile (K = 256) is 1/3 dearer than an oxygen tile
    const int t_beg = tile_at_cost(batch, ((long long)blockIdx.x * batch.cost_total) / gridDim.x);
    const int t_end = blockIdx.x + 1 == gridDim.x ? batch.n_tiles : tile_at_cost(batch, ((long long)(blockIdx.x + 1) * batch.cost_total) / gridDim.x);

    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_aready + 8 * s, 129); // 128 converter threads + the producer's expect_tx for the B tiles
            mbar_init(bar_empty + 8 * s, 1);
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(bar_accf + 8 * b, 1);
            mbar_init(bar_acce + 8 * b, EPI_WARPS * 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

    if (warp == 0) {
        // ===== TMA producer
        if (lane == 0) {
            uint32_t it = 0; // k-block counter across tiles
            for (int t = t_beg; t < t_end; ++t) {
                const TileCoord tc = tile_coord(batch, t);
                const TcGroup &g = batch.g[tc.gi];
                const uint32_t tx_b = (SPLIT3 ? 2u : 1u) * (uint32_t)g.NT * BLOCK_K * 4u;
                const int num_kb = g.K / BLOCK_K;
                for (int kb = 0; kb < num_kb; ++kb, ++it) {
                    const int s = it % S;
                    const uint32_t ph = (it / S) & 1;
                    mbar_wait(bar_empty + 8 * s, ph ^ 1);
                    const uint32_t stage = smem_base + s * stage_bytes;
                    // A -> full[s] (wakes the converters); B -> aready[s], the one barrier the MMA thread waits on
                    mbar_expect_tx(bar_full + 8 * s, A_TILE_BYTES);
                    tma_load_2d(stage, &g.mapA, kb * BLOCK_K, tc.m0, bar_full + 8 * s);
                    mbar_expect_tx(bar_aready + 8 * s, tx_b);
                    tma_load_2d(stage + A_TILE_BYTES, &g.mapBhi, kb * BLOCK_K, tc.n0, bar_aready + 8 * s);
                    if (SPLIT3) tma_load_2d(stage + blo_off, &g.mapBlo, kb * BLOCK_K, tc.n0, bar_aready + 8 * s);
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer: the whole warp runs the loop with warp-uniform values (descriptors stay in uniform
        // registers); one elected lane issues tcgen05.mma / tcgen05.commit.
        {
            uint32_t it = 0;
            int lt = 0; // local tile counter
            for (int t = t_beg; t < t_end; ++t, ++lt) {
                const TileCoord tc = tile_coord(batch, t);
                const TcGroup &g = batch.g[tc.gi];
                const int num_kb = g.K / BLOCK_K;
                const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(g.NT >> 3) << 17) | ((uint32_t)(TILE_M >> 4) << 24);
                const int b = lt & 1;
                const uint32_t acc = tmem_base + (uint32_t)(b * batch.acc_stride);
                mbar_wait(bar_acce + 8 * b, ((lt >> 1) & 1) ^ 1); // epilogue has drained this accumulator buffer
                tc_fence_after();
                for (int kb = 0; kb < num_kb; ++kb, ++it) {
                    const int s = it % S;
                    const uint32_t ph = (it / S) & 1;
                    mbar_wait(bar_aready + 8 * s, ph); // B tiles landed and A converted into TMEM
                    tc_fence_after();
                    const uint32_t stage = smem_base + s * stage_bytes;
                    const uint64_t dhi = make_kmajor_sw128_desc(stage + A_TILE_BYTES);
                    const uint64_t dlo = make_kmajor_sw128_desc(stage + blo_off);
                    const uint32_t a_hi = tmem_base + a_col0 + 64u * (it % (uint32_t)T), a_lo = a_hi + 32;
                    if (elect_one()) {
#pragma unroll
                        for (int k = 0; k < BLOCK_K / UMMA_K; ++k) {
                            const uint64_t koff = (uint64_t)(k * UMMA_K * 4 >> 4);
                            const uint32_t first = (kb | k) ? 1u : 0u;
                            if (SPLIT3) {
                                mma_tf32_ts(acc, a_lo + k * UMMA_K, dhi + koff, idesc, first);
                                mma_tf32_ts(acc, a_hi + k * UMMA_K, dlo + koff, idesc, 1u);
                                mma_tf32_ts(acc, a_hi + k * UMMA_K, dhi + koff, idesc, 1u);
                            } else {
                                mma_tf32_ts(acc, a_hi + k * UMMA_K, dhi + koff, idesc, first);
                            }
                        }
                        tc_commit(bar_empty + 8 * s);
                        if (kb + 1 == num_kb) tc_commit(bar_accf + 8 * b);
                    }
                    __syncwarp();
                }
            }
        }
    } else if (warp < 10) {
        // ===== converters: fp32 A row -> tf32 hi/lo in TMEM.  Two groups of four warps (lane quarters warp & 3)
        // take alternate K blocks, so one block's LDS -> split -> tcgen05.st -> wait latency hides behind the other's.
        const int quarter = warp & 3;
        const int cgroup = (warp - 2) >> 2;
        const int row = quarter * 32 + lane;
        const uint32_t lane_addr = tmem_base + ((uint32_t)(quarter * 32) << 16);
        uint32_t it = 0;
        for (int t = t_beg; t < t_end; ++t) {
            const TileCoord tc = tile_coord(batch, t);
            const int num_kb = batch.g[tc.gi].K / BLOCK_K;
            for (int kb = 0; kb < num_kb; ++kb, ++it) {
                if ((int)(it & 1) != cgroup) continue;
                const int s = it % S;
                const uint32_t ph = (it / S) & 1;
                if (T < S && it >= (uint32_t)T) { // fewer TMEM slots than stages: the slot is free once the MMAs of K block it - T are done
                    const uint32_t jt = it - (uint32_t)T;
                    mbar_wait(bar_empty + 8 * (jt % S), (jt / S) & 1);
                    tc_fence_after();
                }
                mbar_wait(bar_full + 8 * s, ph);
                const uint32_t arow = smem_base + s * stage_bytes + row * 128;
                uint32_t hi[32], lo[32];
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    float4 v;
                    const uint32_t addr = arow + (uint32_t)((c ^ (row & 7)) << 4);
                    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
                    const float x[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const uint32_t h = tf32_round(x[e]);
                        hi[4 * c + e] = h;
                        if (SPLIT3) lo[4 * c + e] = tf32_round(x[e] - __uint_as_float(h));
                    }
                }
                const uint32_t slot = lane_addr + a_col0 + 64u * (it % (uint32_t)T);
                tmem_st32(slot, hi);
                if (SPLIT3) tmem_st32(slot + 32, lo);
                asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                tc_fence_before();
                mbar_arrive(bar_aready + 8 * s);
            }
        }
    } else {
        // ===== epilogue: warps 10..17 -> lane quarters 2,3,0,1,2,3,0,1; this thread owns accumulator row `row`.
        // The accumulator is drained in 16-column chunks; the two warps of a lane quarter take alternate chunks (one warp
        // per quarter could not keep up with the MMAs of a short-K tile: the reverse layers ran at 32 % tensor activity).
        // Global traffic goes through a per-warp 32 x 16 staging chunk so that every LDG/STG covers whole 64-byte row
        // segments (8 rows per instruction).
        const int ew = warp - 10;
        const int quarter = warp & 3;
        const int half = ew >> 2; // parity of the chunks this warp serves
        const int row = quarter * 32 + lane;
        const uint32_t lane_addr = tmem_base + ((uint32_t)(quarter * 32) << 16);
        const uint32_t stg = bar_base + 256 + (uint32_t)ew * EPI_STG_BYTES;
        const uint32_t my_row = stg + (uint32_t)lane * (EPI_STG_LD * 4);
        // cooperative access: 8 rows x 4 x 16 B per instruction; a quarter-warp covers rows q and q + 4, whose staged
        // copies are 80 words apart (bank offset 16): conflict-free with the 20-word row stride
        const int sub_r = (lane >> 3) + 4 * ((lane >> 2) & 1), sub_c = (lane & 3) * 4;
        const float alpha = batch.alpha, inv_alpha = 1.0f / batch.alpha;
        // In-place epilogues read the previous contents of C, written by the forward pass ~200 MB of traffic ago: the row
        // of the NEXT tile this thread owns is pulled into L2 one tile ahead (the two warps of a quarter take alternate
        // lines), so that the chunk loads below see an L2 round trip instead of a DRAM one.
        auto l2_prefetch_tile = [&](int t2) {
            if (!(EPI == EPI_DCELU || EPI == EPI_ACCUM) || t2 >= t_end) return;
            const TileCoord c2 = tile_coord(batch, t2);
            const TcGroup &g2 = batch.g[c2.gi];
            const int m2 = c2.m0 + row;
            if (m2 < g2.M) {
                const char *p2 = reinterpret_cast<const char *>(g2.C + (size_t)m2 * g2.ldc + c2.n0);
                for (int off = half * 128; off < g2.NT * 4; off += 256) asm volatile("prefetch.global.L2 [%0];" ::"l"(p2 + off));
            }
        };
        l2_prefetch_tile(t_beg);
        int lt = 0;
        for (int t = t_beg; t < t_end; ++t, ++lt) {
            const TileCoord tc = tile_coord(batch, t);
            const TcGroup &g = batch.g[tc.gi];
            const int b = lt & 1;
            const int mrow0 = tc.m0 + quarter * 32; // first global row of this warp's 32 rows
            l2_prefetch_tile(t + 1);
            const int m = mrow0 + lane;
            const bool rowok = m < g.M;
            float esum = 0.f;
            // Operands from global memory are fetched one chunk ahead (the L1 is only ~12 KB next to 216 KB of
            // shared memory, so every one of these loads is an L2 round trip): bias / w4 one column per lane
            // (redistributed with shuffles), previous contents 4 x 16 B per lane, coalesced.
            float bias_l = 0.f, w4_l = 0.f;
            float4 pre[4];
            auto prefetch = [&](int c0) {
                if (EPI == EPI_CELU || EPI == EPI_CELU_OUT) bias_l = lane < EPI_CW ? g.bias[tc.n0 + c0 + lane] : 0.f;
                if (EPI == EPI_CELU_OUT) w4_l = lane < EPI_CW ? g.w4[tc.n0 + c0 + lane] : 0.f;
                if (EPI == EPI_DCELU || EPI == EPI_ACCUM) {
                    const float *cb = g.C + (size_t)mrow0 * g.ldc + tc.n0 + c0;
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int r = i * 8 + sub_r;
                        pre[i] = mrow0 + r < g.M ? *reinterpret_cast<const float4 *>(cb + (size_t)r * g.ldc + sub_c)
                                                 : make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                }
            };
            const int c_first = half * EPI_CW;
            if (c_first < g.NT) prefetch(c_first); // before the wait for the accumulator: hides behind the MMAs of this tile
            mbar_wait(bar_accf + 8 * b, (lt >> 1) & 1);
            tc_fence_after();

            for (int c0 = c_first; c0 < g.NT; c0 += 2 * EPI_CW) {
                float *cbase = g.C + (size_t)mrow0 * g.ldc + tc.n0 + c0;
                const float bias_c = bias_l, w4_c = w4_l;
                if (EPI == EPI_DCELU || EPI == EPI_ACCUM) { // previous contents -> staging
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int r = i * 8 + sub_r;
                        asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(stg + (uint32_t)(r * EPI_STG_LD + sub_c) * 4), "f"(pre[i].x), "f"(pre[i].y), "f"(pre[i].z), "f"(pre[i].w) : "memory");
                    }
                    __syncwarp();
                }
                if (c0 + 2 * EPI_CW < g.NT) prefetch(c0 + 2 * EPI_CW);
                uint32_t acc[16];
                tmem_ld16(lane_addr + (uint32_t)(b * batch.acc_stride) + c0, acc);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int col = 4 * q;
                    float4 o;
                    float *ov = reinterpret_cast<float *>(&o);
                    float4 prev = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (EPI == EPI_DCELU || EPI == EPI_ACCUM)
                        asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(prev.x), "=f"(prev.y), "=f"(prev.z), "=f"(prev.w) : "r"(my_row + col * 4));
                    const float *pv = reinterpret_cast<const float *>(&prev);
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        float v = __uint_as_float(acc[4 * q + e]);
                        float bv = 0.f, wv = 0.f;
                        if (EPI == EPI_CELU || EPI == EPI_CELU_OUT) bv = __shfl_sync(0xffffffffu, bias_c, col + e);
                        if (EPI == EPI_CELU_OUT) wv = __shfl_sync(0xffffffffu, w4_c, col + e);
                        if (EPI == EPI_CELU) v = celu_fwd(v + bv, alpha, inv_alpha);
                        if (EPI == EPI_CELU_OUT) {
                            const float hh = celu_fwd(v + bv, alpha, inv_alpha);
                            esum = fmaf(hh, wv, esum);
                            v = wv * celu_grad_from_h(hh, inv_alpha);
                        }
                        if (EPI == EPI_DCELU) v *= celu_grad_from_h(pv[e], inv_alpha);
                        if (EPI == EPI_ACCUM) v += pv[e];
                        ov[e] = v;
                    }
                    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(my_row + col * 4), "f"(o.x), "f"(o.y), "f"(o.z), "f"(o.w) : "memory");
                }
                __syncwarp();
#pragma unroll
                for (int i = 0; i < 4; ++i) { // staging -> global, whole 64-byte row segments
                    const int r = i * 8 + sub_r;
                    if (mrow0 + r < g.M) {
                        float4 v;
                        asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(stg + (uint32_t)(r * EPI_STG_LD + sub_c) * 4));
                        if (EPI == EPI_RED) atomicAdd(reinterpret_cast<float4 *>(cbase + (size_t)r * g.ldc + sub_c), v); // RED.ADD.F32x4
                        else *reinterpret_cast<float4 *>(cbase + (size_t)r * g.ldc + sub_c) = v;
                    }
                }
                __syncwarp();
            }
            // the accumulator buffer may be overwritten by the MMAs of tile lt + 2
            tc_fence_before();
            mbar_arrive(bar_acce + 8 * b);
            // every epilogue warp (both chunk parities, each n-part of a wide layer) adds its share of the output-layer dot
            if (EPI == EPI_CELU_OUT && rowok) atomicAdd(g.e_atom + m, esum);
        }
    }
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
    }
}

// ---------------------------------------------------------------- host side
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

// 2-D fp32 tensor [rows][cols] with row pitch `ld` floats; box = [box_rows][32 cols], 128-byte swizzle, zero fill
bool make_map(CUtensorMap *m, const float *base, int rows, int cols, int ld, int box_rows)
{
    cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)ld * 4};
    cuuint32_t box[2] = {(cuuint32_t)BLOCK_K, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    return g_encode(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void *)base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int g_num_sms = 0;

template <int EPI>
void launch(cudaStream_t st, const TcBatch &b, int tiles, bool split3)
{
    if (!g_num_sms) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&g_num_sms, cudaDevAttrMultiProcessorCount, dev);
        if (g_num_sms <= 0) g_num_sms = 148;
    }
    const int grid = tiles < g_num_sms ? tiles : g_num_sms; // persistent: one CTA per SM
    const int smem = b.stages * b.stage_bytes + SMEM_FIXED;
    if (split3) {
        cudaFuncSetAttribute(k_gemm_tc<EPI, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_LIMIT);
        k_gemm_tc<EPI, true><<<grid, THREADS, smem, st>>>(b);
    } else {
        cudaFuncSetAttribute(k_gemm_tc<EPI, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_LIMIT);
        k_gemm_tc<EPI, false><<<grid, THREADS, smem, st>>>(b);
    }
}

} // namespace

int nnp_launch_gemm_tc(nnp_ctx *c, const GemmBatch &b, int epi, int split3)
{
    if (!load_encode()) { c->err = "cuTensorMapEncodeTiled entry point not available"; return NNP_ECUDA; }
    TcBatch tb;
    memset(&tb, 0, sizeof(tb));
    tb.alpha = b.alpha;
    int tiles = 0, nt_max = 16;
    // Full-width tiles (one A load and conversion per 128 rows) where every group of the launch fits in 192 columns;
    // a launch with a wider layer splits it into <= 128-column parts, and then the 48 KiB stages / 4-deep ring serve
    // all its groups better than 64 KiB stages / 3-deep (measured on the 98k water box: 0.363 -> 0.344 ms over the six GEMMs)
    int nt_cap = NT_MAX;
    const int tile_fixed = 3000; // fixed cost of a tile in the balance below, in 128-byte units
    for (int i = 0; i < b.n_groups; ++i)
        if (b.g[i].N > NT_MAX) nt_cap = 128;
    for (int i = 0; i < b.n_groups; ++i) {
        const GemmGroup &g = b.g[i];
        TcGroup &t = tb.g[i];
        if (!g.Bt_hi || !g.Bt_lo) { c->err = "tensor-core path: weight operand has no tf32 split"; return NNP_EINVAL; }
        int NT = g.N;                       // <= 192 columns per tile; wider layers in equal parts that are multiples of 16
        int parts = 1;
        while (NT > nt_cap || (g.N % parts) || (NT % 16)) {
            ++parts;
            if (parts > 64) { c->err = "tensor-core path: unsupported GEMM width"; return NNP_EINVAL; }
            NT = g.N / parts;
        }
        if (g.K % BLOCK_K) { c->err = "tensor-core path: K must be a multiple of 32"; return NNP_EINVAL; }
        if (!make_map(&t.mapA, g.A, g.M, g.K, g.lda, TILE_M) || !make_map(&t.mapBhi, g.Bt_hi, g.N, g.K, g.K, NT) ||
            !make_map(&t.mapBlo, g.Bt_lo, g.N, g.K, g.K, NT)) {
            c->err = "cuTensorMapEncodeTiled failed";
            return NNP_ECUDA;
        }
        t.C = g.C; t.bias = g.bias; t.w4 = g.w4; t.e_atom = g.e_atom;
        t.M = g.M; t.N = g.N; t.K = g.K; t.ldc = g.ldc;
        t.NT = NT;
        t.n_tiles_n = g.N / NT;
        if (NT > nt_max) nt_max = NT;
        tb.tile_off[i] = tiles;
        tiles += nnp_div_up(g.M, TILE_M) * t.n_tiles_n;
        // bytes through the SM in units of 128 B (the kernel is bound by L2 -> SM traffic): per K block the A tile and the
        // hi/lo weight tiles, plus the output tile (read and written by the in-place epilogues)
        // ... plus a fixed 3000 per tile for the pipeline fill / accumulator hand-over (swept 0..20000 on the 98k water box with the
        // eight-warp epilogue: the six GEMMs take 0.323 ms at 1000, 0.314 at 3000, 0.313 at 4000, 0.329 at 8000; the layers
        // move in steps of ~4 us as the slowest CTA gains or loses a tile, which a dynamic tile queue would even out)
        tb.tile_cost[i] = g.K / BLOCK_K * (TILE_M + 2 * NT) + ((epi == EPI_DCELU || epi == EPI_ACCUM) ? 8 : 4) * NT + tile_fixed;
        tb.cost_total += (long long)tb.tile_cost[i] * (tiles - tb.tile_off[i]);
    }
    tb.n_groups = b.n_groups;
    tb.tile_off[b.n_groups] = tiles;
    tb.n_tiles = tiles;
    if (tiles == 0) return NNP_OK;
    tb.b_tile_bytes = nt_max * BLOCK_K * 4;
    tb.stage_bytes = A_TILE_BYTES + 2 * tb.b_tile_bytes;       // multiples of 1 KiB: swizzle atoms stay aligned
    tb.stages = (SMEM_LIMIT - SMEM_FIXED) / tb.stage_bytes;
    if (tb.stages > STAGES_MAX) tb.stages = STAGES_MAX;
    tb.acc_stride = nt_max <= 128 ? 128 : 192;
    tb.a_slots = (TMEM_COLS - 2 * tb.acc_stride) / 64;
    if (tb.a_slots > tb.stages) tb.a_slots = tb.stages;
    const bool s3 = split3 != 0;
    switch (epi) {
    case EPI_CELU: launch<EPI_CELU>(c->stream, tb, tiles, s3); break;
    case EPI_CELU_OUT: launch<EPI_CELU_OUT>(c->stream, tb, tiles, s3); break;
    case EPI_DCELU: launch<EPI_DCELU>(c->stream, tb, tiles, s3); break;
    case EPI_STORE: launch<EPI_STORE>(c->stream, tb, tiles, s3); break;
    case EPI_ACCUM: launch<EPI_ACCUM>(c->stream, tb, tiles, s3); break;
    case EPI_RED: launch<EPI_RED>(c->stream, tb, tiles, s3); break;
    default: c->err = "bad epilogue"; return NNP_EINVAL;
    }
    c->launches += 1;
    return NNP_OK;
}
