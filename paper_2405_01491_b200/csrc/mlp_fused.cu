// Stage 3 + the MLP half of stage 4 as ONE persistent kernel (mm_mode NNP_MM_3XF16_TC): a CTA owns a 128-atom row tile
// and takes it through the whole chain  G -> h1 -> h2 -> h3 (-> e_i, delta3) -> delta2 -> delta1 -> dE/dG  without
// leaving the SM (ChemicalNet; forces by reverse mode, L65 / L176; the model of Fig. 2 is one fused
// executable, L176).  SURVEY.md 8(f)-4 / 8(d) "intermediates": the unfused path (mlp_tc.cu, six launches) writes and
// re-reads every activation through HBM (~0.8 GB per step on the 98k water box) and pays six launch / pipeline-fill costs.
//
// Arithmetic ("3xF16"): every fp32 operand x is split into hi = fp16(x) and lo = fp16(x - hi) (11 + 11 significant bits,
// the same widths as the tf32 split of mlp_tc.cu) and A.B is accumulated in fp32 by tcgen05.mma kind::f16 as
// A_lo.B_hi + A_hi.B_lo + A_hi.B_hi.  fp16 has the narrow exponent: weights are scaled per matrix by a power of two so
// that max |w| lands in [2^13, 2^14), activations by 2^4; both scalings are undone exactly in the epilogue.  A value
// above 60000 after scaling (|activation| > 3750) raises NNP_FLAG_RANGE -> NNP_ERANGE instead of silently saturating.
//
// How a layer feeds the next one - IN PLACE in tensor memory.  TMEM holds two 256-column regions.  The accumulator of
// GEMM j ([128 atoms] x [N_j], fp32) lives in one of them.  When its last MMA has completed, sixteen epilogue warps drain
// it 16 columns at a time: bias + CELU (forward) or x CELU'(h) (reverse), split into fp16 hi / lo - and the 16 fp32
// columns just read are exactly the room their own hi (8 columns of packed pairs) and lo (8 columns) need as the A
// operand of GEMM j+1, so the chunk is written back where it came from (tcgen05.st) and its mbarrier is armed.  The MMA
// thread multiplies each chunk with the matching 16 rows of W_{j+1} as soon as it is ready (tcgen05.mma .ts form: A from
// TMEM, B = weight tile in shared memory) into the OTHER region: no operand ring, no slot recycling, the epilogue never
// waits for the tensor pipe.  Nothing but the weights is streamed: they are pre-packed at set-up into the exact
// 128-byte-swizzled K-major fp16 tile images the MMA descriptors expect ([K block of 64][part][hi | lo][rows][64]), one
// tile = one contiguous cp.async.bulk of up to 32 KiB into a ring of shared-memory entries.
//   h1 and h2 are needed again by the reverse layers (CELU' = 1 + min(h,0)/alpha).  They do not fit on the SM next to the
// weight ring, so the forward epilogues also write them to the activation buffers and the reverse epilogues of the same
// CTA read them back a few microseconds later (L2 hits; 1.8 KB per atom and direction).
//
// One chain for every system: F1 F2 F3 B3 B2 B1, input G (TMA), output dE/dG.  With more than 256 active AEV columns (e.g.
// 1024 for seven species) the first and the last GEMM are wider than a TMEM region: F1 takes its operand through the region in
// passes of 16 chunks (a slot is rewritten once the MMAs of the pass before have completed), B1 writes its output in passes of
// 256 columns into the same region, from the operand that stays in the other one (kernels with WIDE = true).
// Warp roles: 0 producer (TMA tiles of the chain's input + bulk weight copies), 1 and 18 MMA issue (even / odd chunks),
// 2-17 epilogue (four warps per TMEM lane quarter, every fourth 16-column chunk each); the epilogue warps also convert the
// chain's input (fp32 tile in shared memory -> fp16 hi / lo chunks in TMEM) at the start of a tile.  608 threads, at most
// five warps per SM quadrant: 96 registers each - with ~200 KiB of the SM's 228 KiB configured as shared memory,
// local-memory traffic would go to L2.
#include <cuda.h>
#include <cuda_fp16.h>

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "nnp_internal.cuh"

namespace {

#include "tc_ptx.cuh"

constexpr int TILE_M = 128;
constexpr int KBH = 64;                // K block of the weight tiles: fp16 elements of one 128-byte swizzle row
constexpr int KBF = 32;                // K block of the input tiles: fp32 elements of one 128-byte swizzle row
constexpr int CH = 16;                 // K chunk: one tcgen05.mma kind::f16 K step, 16 accumulator columns
constexpr int MAX_STAGES = 6;
constexpr int NW = 4;                  // weight ring entries
constexpr int W_ENTRY_BYTES = 32768;   // hi + lo tiles of up to 128 rows x 128 B
constexpr int NA = 2;                  // ring of input tiles
constexpr int A_TILE_BYTES = TILE_M * KBF * 4;
constexpr int EPI_WARPS = 16;
constexpr int EPI_SETS = EPI_WARPS / 4;
constexpr int EPI_STG_LD = 20;
constexpr int EPI_STG_BYTES = 32 * EPI_STG_LD * 4;
constexpr int BAR_BYTES = 512;
constexpr int GCACHE = 8;               // group descriptors a CTA keeps in shared memory (its tile range spans at most that many)
constexpr int GROUP_BYTES = 576;
constexpr int SB_BYTES = 4 * 256 * 4;     // biases of the three forward GEMMs (x 16) and w4 of the current group
constexpr int SMEM_BYTES = 1024 + NW * W_ENTRY_BYTES + NA * A_TILE_BYTES + BAR_BYTES + EPI_WARPS * EPI_STG_BYTES + GCACHE * GROUP_BYTES + SB_BYTES;
constexpr int MMA2_WARP = 2 + EPI_WARPS;  // the second MMA-issuing warp (odd chunks)
constexpr int THREADS = (3 + EPI_WARPS) * 32;
constexpr int REGION_COLS = 256;       // two accumulator / operand regions: columns [0, 256) and [256, 512)
constexpr int GRP = 4 * CH;                // columns per round of the epilogue: one chunk of every set, one K block of weights
constexpr int MAX_CHUNKS = REGION_COLS / CH;
constexpr int ACT_SHIFT = 4;           // activations enter the tensor core multiplied by 2^4
constexpr float ACT_SCALE = 16.0f;
constexpr float RANGE_LIMIT = 60000.0f;
static_assert(SMEM_BYTES <= 227 * 1024, "shared memory budget");
static_assert(NA == 2, "input tile k lives in ring entry k & 1: one entry per pair of epilogue sets");
static_assert(8 * (2 * NW + 2 * NA + 2 * MAX_CHUNKS + 2 + 4) + 8 <= BAR_BYTES, "barrier area");

enum FusedEpi {
    FE_FWD = 0,     // h = celu(acc + bias): stash h, hi/lo -> operand
    FE_OUT = 1,     // h3 = celu(acc + bias); e_atom += h3 . w4; delta3 = w4 celu'(h3): hi/lo -> operand
    FE_BWD = 2,     // delta = acc * celu'(stash): hi/lo -> operand
    FE_ST = 3,      // out = acc
    FE_RED = 4      // out += acc (vector reductions in memory: ensembles add into the same rows)
};

struct FusedStage {
    int K, N;            // K: columns of the A operand (multiple of 32); N: output columns (multiple of 32, <= 256)
    int epi;
    uint32_t w_off;      // byte offset of the packed weight tiles of this GEMM in the blob
    const float *bias;   // [N] forward GEMMs: bias * 2^ACT_SHIFT
    float *stash;        // rows of 16 h: written by FE_FWD, read by FE_BWD (already offset to the group's first row)
    int ld_stash;
    int brow;            // forward GEMMs: row of the shared-memory bias table
    float c_acc;         // forward: acc -> 16 z;  FE_ST / FE_RED: acc -> true value
    float gs, gc;        // reverse: out = acc * fma(min(h, 0), gs, gc)  (the scalings folded into CELU')
    int n_total;         // output columns in all: > N for the last GEMM of a wide chain, which runs in passes of N columns
};

struct alignas(64) FusedGroup {
    CUtensorMap mapA;    // input of the chain: [M][K0] fp32, row pitch of the source buffer
    const uint8_t *wblob;
    const float *w4;
    float *e_atom;
    float *out;          // output rows of the last GEMM
    int ldo;
    int M, n_stages, tile0, n_tiles;
    int h3;              // width of the last hidden layer (length of w4)
    int pad_[14];
    FusedStage st[MAX_STAGES];
};

static_assert(sizeof(FusedGroup) == GROUP_BYTES, "group descriptor size");

__device__ __forceinline__ void bulk_load(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar)
                 : "memory");
}

// D[tmem] (+)= A[tmem] . B[smem desc]^T, kind::f16 (fp16 operands, fp32 accumulate), A from tensor memory
__device__ __forceinline__ void mma_f16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),
        "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}

__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[16])
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
        "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
        "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
        : "memory");
}

// Packed fp32 pairs (FFMA2 / FMUL2 / FADD2): one issue slot for two columns of the epilogue arithmetic.
__device__ __forceinline__ float2 f2_fma(const float2 a, const float2 b, const float2 c)
{
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;"
        : "=l"(d)
        : "l"(*reinterpret_cast<const unsigned long long *>(&a)), "l"(*reinterpret_cast<const unsigned long long *>(&b)),
          "l"(*reinterpret_cast<const unsigned long long *>(&c)));
    return *reinterpret_cast<float2 *>(&d);
}
__device__ __forceinline__ float2 f2_mul(const float2 a, const float2 b)
{
    unsigned long long d;
    asm("mul.rn.f32x2 %0, %1, %2;"
        : "=l"(d)
        : "l"(*reinterpret_cast<const unsigned long long *>(&a)), "l"(*reinterpret_cast<const unsigned long long *>(&b)));
    return *reinterpret_cast<float2 *>(&d);
}
__device__ __forceinline__ float2 f2_add(const float2 a, const float2 b)
{
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;"
        : "=l"(d)
        : "l"(*reinterpret_cast<const unsigned long long *>(&a)), "l"(*reinterpret_cast<const unsigned long long *>(&b)));
    return *reinterpret_cast<float2 *>(&d);
}
__device__ __forceinline__ float2 f2_bc(const float s) { return make_float2(s, s); }

// 16 consecutive K values of one row -> the row's 16 operand columns: hi pairs (k, k+1) in columns 0..7, lo pairs in 8..15
__device__ __forceinline__ void split16(const float (&x)[16], uint32_t (&v)[16])
{
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const __half2 h = __floats2half2_rn(x[2 * q], x[2 * q + 1]);
        const float2 hf = __half22float2(h);
        const float2 lf = f2_fma(hf, f2_bc(-1.0f), make_float2(x[2 * q], x[2 * q + 1])); // x - hi, exact
        const __half2 l = __floats2half2_rn(lf.x, lf.y);
        v[q] = *reinterpret_cast<const uint32_t *>(&h);
        v[8 + q] = *reinterpret_cast<const uint32_t *>(&l);
    }
}

__device__ __forceinline__ int find_group(const FusedGroup *__restrict__ groups, int n_groups, int t)
{
    int gi = 0;
    while (gi + 1 < n_groups && t >= groups[gi + 1].tile0) ++gi;
    return gi;
}

// One accumulator through one epilogue warp: the 16-column chunks set, set + 4, ... of the warp's 32 rows.
// lane_set = lane | set << 8, accf = accumulator barrier address | parity << 31; returns (max |operand value|, row's
// partial energy sum).  Inlined once per GEMM of a chain (the kernel is specialised per chain, below): as functions called
// from a loop over the stages, the caller's state went through local memory around every call - which on this kernel is L2.
template <int EPI>
__device__ __forceinline__ float2 epi_stage(const FusedGroup *gp, int j, int mrow0, int lane_set, uint32_t tm_acc, uint32_t stg,
                                         uint32_t accf, uint32_t bar_ready, uint32_t sb, float alpha, int aux, int n_cols, int col_off)
{
    float vmax = 0.f;
    float2 esum = make_float2(0.f, 0.f);
    constexpr bool fwd = EPI == FE_FWD || EPI == FE_OUT;
    constexpr bool rd_prev = EPI == FE_BWD;                        // reads rows of h for CELU'
    constexpr bool to_op = EPI == FE_FWD || EPI == FE_OUT || EPI == FE_BWD;
    constexpr bool wr_rows = EPI == FE_FWD || EPI == FE_ST || EPI == FE_RED;
    const FusedGroup &g = *gp;
    const FusedStage &st = g.st[j];
    const int lane = lane_set & 31;
    const int N = n_cols, M = g.M; // columns of this accumulator (a pass of the last GEMM of a wide chain: col_off onwards)
    const uint32_t my_row = stg + (uint32_t)lane * (EPI_STG_LD * 4);
    const int sub_r = (lane >> 3) + 4 * ((lane >> 2) & 1), sub_c = (lane & 3) * 4;
    // rows read (h for CELU') and rows written (h stash, or the chain's output)
    const float *rd_base = st.stash;
    const int rd_ld = st.ld_stash;
    float *wr_base = EPI == FE_FWD ? st.stash : g.out + col_off;
    const int wr_ld = EPI == FE_FWD ? st.ld_stash : g.ldo;
    const float c_acc = st.c_acc, gs = st.gs, gc = st.gc;
    // everything the chunk loop needs sits in registers: the "memory" clobbers of the asm statements below would make the
    // compiler re-read any field it still reaches through a pointer, once per chunk
    const uint32_t sbias = sb + (uint32_t)st.brow * (REGION_COLS * 4), sw4 = sb + 3u * (REGION_COLS * 4);
    const int c_first = (lane_set >> 8) * CH;
    const float inv_alpha = 1.0f / alpha;
    const float a16 = alpha * ACT_SCALE;                               // 16 h = max(16 z, 0) + 16 alpha (e - 1)
    const float ce = 1.4426950408889634f / (alpha * ACT_SCALE);       // e = 2^(min(16 z, 0) ce)
    float4 pre[4];
    auto prefetch = [&](int c0) {
        const float *cb = rd_base + (size_t)mrow0 * rd_ld + c0;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int r = i * 8 + sub_r;
            pre[i] = mrow0 + r < M ? *reinterpret_cast<const float4 *>(cb + (size_t)r * rd_ld + sub_c) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
    };
    if (rd_prev && c_first < N) prefetch(c_first);
    mbar_wait(accf & 0x7fffffffu, accf >> 31, 400 + j, aux);
    tc_fence_after();
    for (int c0 = c_first; c0 < N; c0 += GRP) {
        uint32_t a[16];
        tmem_ld16(tm_acc + (uint32_t)c0, a);
        if (rd_prev) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int r = i * 8 + sub_r;
                asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(stg + (uint32_t)(r * EPI_STG_LD + sub_c) * 4), "f"(pre[i].x), "f"(pre[i].y), "f"(pre[i].z), "f"(pre[i].w) : "memory");
            }
            __syncwarp();
            if (c0 + GRP < N) prefetch(c0 + GRP);
        }
        float ov[16];
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            float4 x4 = make_float4(0.f, 0.f, 0.f, 0.f), w4v = make_float4(0.f, 0.f, 0.f, 0.f);
            if (fwd) asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(x4.x), "=f"(x4.y), "=f"(x4.z), "=f"(x4.w) : "r"(sbias + (uint32_t)(c0 + 4 * q) * 4));
            if (EPI == FE_OUT) asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(w4v.x), "=f"(w4v.y), "=f"(w4v.z), "=f"(w4v.w) : "r"(sw4 + (uint32_t)(c0 + 4 * q) * 4));
            if (rd_prev) asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(x4.x), "=f"(x4.y), "=f"(x4.z), "=f"(x4.w) : "r"(my_row + q * 16));
            const float xq[4] = {x4.x, x4.y, x4.z, x4.w};
            const float wq[4] = {w4v.x, w4v.y, w4v.z, w4v.w};
#pragma unroll
            for (int e = 0; e < 4; e += 2) { // two columns at a time: packed fp32 arithmetic, min / max and ex2 per column
                float2 v = make_float2(__uint_as_float(a[4 * q + e]), __uint_as_float(a[4 * q + e + 1]));
                const float2 x2 = make_float2(xq[e], xq[e + 1]);
                if (fwd) {
                    const float2 z = f2_fma(v, f2_bc(c_acc), x2);
                    const float2 t = f2_mul(make_float2(fminf(z.x, 0.f), fminf(z.y, 0.f)), f2_bc(ce));
                    float2 ex;
                    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(ex.x) : "f"(t.x));
                    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(ex.y) : "f"(t.y));
                    v = f2_fma(f2_bc(a16), ex, f2_add(make_float2(fmaxf(z.x, 0.f), fmaxf(z.y, 0.f)), f2_bc(-a16))); // 16 h
                    if (EPI == FE_OUT) {
                        const float2 w2 = make_float2(wq[e], wq[e + 1]);
                        esum = f2_fma(v, w2, esum);
                        v = f2_mul(w2, f2_fma(make_float2(fminf(v.x, 0.f), fminf(v.y, 0.f)), f2_bc(inv_alpha), f2_bc(ACT_SCALE))); // 16 w4 celu'(h3)
                    }
                } else if (rd_prev) {
                    v = f2_mul(v, f2_fma(make_float2(fminf(x2.x, 0.f), fminf(x2.y, 0.f)), f2_bc(gs), f2_bc(gc)));
                } else {
                    v = f2_mul(v, f2_bc(c_acc));
                }
                ov[4 * q + e] = v.x;
                ov[4 * q + e + 1] = v.y;
            }
        }
        if (to_op) {
            uint32_t sl[16];
#pragma unroll
            for (int q = 0; q < 16; ++q) vmax = fmaxf(vmax, fabsf(ov[q]));
            split16(ov, sl);
            tmem_st16(tm_acc + (uint32_t)c0, sl); // hi / lo of the chunk go back into the accumulator's own columns
        }
        if (wr_rows) {
#pragma unroll
            for (int q = 0; q < 4; ++q)
                asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(my_row + q * 16), "f"(ov[4 * q]), "f"(ov[4 * q + 1]), "f"(ov[4 * q + 2]), "f"(ov[4 * q + 3]) : "memory");
        }
        if (to_op) {
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            tc_fence_before();
        }
        __syncwarp();
        if (to_op && lane == 0) mbar_arrive(bar_ready + 8 * (c0 / CH));
        if (wr_rows) {
            float *cbase = wr_base + (size_t)mrow0 * wr_ld + c0;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int r = i * 8 + sub_r;
                if (mrow0 + r < M) {
                    float4 v;
                    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(stg + (uint32_t)(r * EPI_STG_LD + sub_c) * 4));
                    if (EPI == FE_RED) atomicAdd(reinterpret_cast<float4 *>(cbase + (size_t)r * wr_ld + sub_c), v);
                    else *reinterpret_cast<float4 *>(cbase + (size_t)r * wr_ld + sub_c) = v;
                }
            }
            __syncwarp();
        }
    }
    return make_float2(vmax, esum.x + esum.y);
}

// rows of the two MMAs of a GEMM with N columns: 128 + (N - 128), or N alone (one MMA with N > 128 and its operand in
// tensor memory ran at a quarter of the rate of two with N <= 128: measured, 370 against 2 x 64 cycles at N = 192)
__device__ __forceinline__ int part_rows(int N, int p) { return p == 0 ? (N > 128 ? 128 : N) : N - 128; }

// Regions alternate along the chain AND across tiles: a running count rc of operand generations (the chain input is
// generation rc, the accumulator of GEMM j generation rc + 1 + j, the next tile starts at rc + n_stages + 1) gives
// generation q the region q & 1, so the input of tile t+1 goes where the last GEMM of tile t took its operand from while
// the last accumulator of tile t is still being drained from the other one.

// Chains (template parameter of the kernel): 0 one network (dE/dG stored), 1 ensemble (dE/dG accumulated with reductions).
enum { CHAIN_FULL = 0, CHAIN_FULL_RED = 1 };
__host__ __device__ constexpr int chain_len(int) { return 6; }
__host__ __device__ constexpr int chain_epi(int chain, int j)
{
    return j < 2 ? FE_FWD : j == 2 ? FE_OUT : j < 5 ? FE_BWD : chain == CHAIN_FULL_RED ? FE_RED : FE_ST;
}

// WIDE: the chain's input / output has more than 256 columns (first GEMM: operand passes, last GEMM: output passes); the
// narrow kernels carry none of the pass logic.
template <int CHAIN, bool WIDE>
__global__ void __launch_bounds__(THREADS, 1)
k_mlp_fused(const FusedGroup *__restrict__ groups, int n_groups, const int *__restrict__ cta_tiles, float alpha, int *__restrict__ flags)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t w_ring = smem_base, a_ring = smem_base + NW * W_ENTRY_BYTES;
    const uint32_t bar_base = a_ring + NA * A_TILE_BYTES;
    // barriers (8 B each)
    const uint32_t bar_wfull = bar_base, bar_wempty = bar_base + 8 * NW;
    const uint32_t bar_afull = bar_base + 16 * NW, bar_aempty = bar_afull + 8 * NA;
    const uint32_t bar_ready = bar_aempty + 8 * NA;            // [2 regions][MAX_CHUNKS]: operand chunk written
    const uint32_t bar_accf = bar_ready + 8 * 2 * MAX_CHUNKS;  // [2 regions]: every MMA into the region has completed
    const uint32_t bar_drained = bar_accf + 16;                // an accumulator of the chain's last GEMM has been read
    const uint32_t bar_pass = bar_drained + 8;                 // wide input: the MMAs of a pass of 16 chunks have completed
    const uint32_t bar_first = bar_pass + 8;                   // the MMAs of chunk 0 of a GEMM (they overwrite the accumulator) have completed
    const uint32_t tmem_slot = bar_first + 8;
    const uint32_t stg_base = bar_base + BAR_BYTES;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int t_beg = cta_tiles[blockIdx.x], t_end = cta_tiles[blockIdx.x + 1];
    // The descriptors of the groups this CTA's tiles belong to go to shared memory once: with ~200 KiB of the SM carved
    // out as shared memory the L1 holds next to nothing, and every field read from the table in global memory was an L2
    // round trip on the critical path of a stage.  (The tensor map is used from its place in global memory.)
    const uint32_t sb_base = stg_base + EPI_WARPS * EPI_STG_BYTES + GCACHE * GROUP_BYTES;
    const FusedGroup *gsm = reinterpret_cast<const FusedGroup *>(smem_raw + (stg_base + EPI_WARPS * EPI_STG_BYTES - smem_u32(smem_raw)));
    const int g_lo = t_beg < t_end ? find_group(groups, n_groups, t_beg) : 0;
    const int n_gc = t_beg < t_end ? find_group(groups, n_groups, t_end - 1) - g_lo + 1 : 0;
    {
        const uint4 *src = reinterpret_cast<const uint4 *>(groups + g_lo);
        uint4 *dst = reinterpret_cast<uint4 *>(const_cast<FusedGroup *>(gsm));
        for (int k = threadIdx.x; k < n_gc * (GROUP_BYTES / 16); k += THREADS) dst[k] = src[k];
    }

    if (threadIdx.x == 0) {
        for (int e = 0; e < NW; ++e) { mbar_init(bar_wfull + 8 * e, 1); mbar_init(bar_wempty + 8 * e, 2); } // (both MMA warps release an entry)
        for (int e = 0; e < NA; ++e) { mbar_init(bar_afull + 8 * e, 1); mbar_init(bar_aempty + 8 * e, 8); }
        for (int k = 0; k < 2 * MAX_CHUNKS; ++k) mbar_init(bar_ready + 8 * k, 4);
        mbar_init(bar_accf, 2);
        mbar_init(bar_accf + 8, 2);
        mbar_init(bar_drained, EPI_WARPS);
        mbar_init(bar_pass, 2);
        mbar_init(bar_first, 1);
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
        // ===== producer: everything that arrives in shared memory.  Weights in their order of use; the first NA input tiles
        // of the NEXT tile are requested while this tile is in its third GEMM (their ring entries are free by then), so that
        // the conversion at the start of a tile never waits for a load queued behind the whole weight stream.
        if (lane == 0) {
            uint32_t wi = 0, aph0 = 0, aph1 = 0; // phases of the two input-ring entries requested so far
            int pre = 0; // input tiles of tile t already requested
            for (int t = t_beg; t < t_end; ++t) {
                const int gi = find_group(gsm, n_gc, t);
                const FusedGroup &g = gsm[gi];
                const int m0 = (t - g.tile0) * TILE_M;
                const int n_stages = g.n_stages;
                // Input tile k of a row tile always goes to ring entry k & 1: even tiles (chunks 4i, 4i + 1) are read by the
                // epilogue sets 0 and 1, odd tiles by sets 2 and 3, so every entry has ONE group of readers that takes each
                // of its phases in turn.  (An mbarrier wait names a phase by its parity only: a reader that skipped a phase
                // of an entry - with a ring of three the set pairs alternated on each entry - takes the phase before for its
                // own and reads a tile that has not arrived; found as rare wrong energies and a hang on a wide chain.)
                auto load_a = [&](const FusedGroup &gg, int gidx, int row0, int k) {
                    const uint32_t e = (uint32_t)k & 1u;
                    uint32_t &ph = e ? aph1 : aph0;
                    mbar_wait(bar_aempty + 8 * e, (ph & 1u) ^ 1u, 150, k);
                    mbar_expect_tx(bar_afull + 8 * e, A_TILE_BYTES);
                    tma_load_2d(a_ring + e * A_TILE_BYTES, &groups[g_lo + gidx].mapA, k * KBF, row0, bar_afull + 8 * e);
                    ++ph;
                };
                int a_next = pre; // next input tile (32 columns) of this tile to request
                pre = 0;
                for (int j = 0; j < n_stages; ++j) {
                    const int K = g.st[j].K, Np = g.st[j].N;
                    const int n_total = (WIDE && j + 1 == n_stages) ? g.st[j].n_total : Np;
                    const uint8_t *wsrc = g.wblob + g.st[j].w_off; // the passes of a wide last GEMM are packed one after the other
                    if (j == 2 && t + 1 < t_end) {
                        const int gn = find_group(gsm, n_gc, t + 1);
                        const FusedGroup &g2 = gsm[gn];
                        const int nka = g2.st[0].K / KBF;
                        for (; pre < NA && pre < nka; ++pre) load_a(g2, gn, (t + 1 - g2.tile0) * TILE_M, pre);
                    }
                    for (int col = 0; col < n_total; col += Np) {
                        const int N = n_total - col < Np ? n_total - col : Np;
                        for (int kb = 0; kb < (K + KBH - 1) / KBH; ++kb) {
                            if (j == 0)
                                for (; a_next < 2 * kb + 2 && a_next * KBF < K; ++a_next) load_a(g, gi, m0, a_next);
                            for (int p = 0; p < (N > 128 ? 2 : 1); ++p, ++wi) {
                                const uint32_t e = wi % NW;
                                const uint32_t bytes = 2u * (uint32_t)part_rows(N, p) * 128u; // hi tile, lo tile behind it
                                mbar_wait(bar_wempty + 8 * e, ((wi / NW) & 1) ^ 1, 100 + j, (t - t_beg) * 100 + kb);
                                mbar_expect_tx(bar_wfull + 8 * e, bytes);
                                bulk_load(w_ring + e * W_ENTRY_BYTES, wsrc, bytes, bar_wfull + 8 * e);
                                wsrc += bytes;
                            }
                        }
                    }
                }
            }
        }
    } else if (warp == 1 || warp == MMA2_WARP) {
        // ===== MMA issue (two warps).  The whole warp walks the loop and one elected lane issues; every value an MMA takes is first made
        // PROVABLY warp-uniform (uni(): a broadcast from lane 0) - the operands of tcgen05.mma live in uniform registers, and
        // for values the compiler cannot prove uniform (anything loaded from memory) it wraps each MMA in an
        // elect / R2UR.BROADCAST loop of a dozen dependent instructions (~150 cycles per MMA measured).
        auto uni = [](uint32_t v) { return __shfl_sync(0xffffffffu, v, 0); };
        const uint32_t tb = uni(tmem_base), wr = uni(w_ring);
        const int tu_beg = (int)uni((uint32_t)t_beg), tu_end = (int)uni((uint32_t)t_end);
        // Two warps issue: this one (mw = 0) the even chunks of every GEMM, the second (mw = 1) the odd ones.  Waiting for a
        // chunk, electing a lane and moving an MMA's operands into uniform registers costs ~500 cycles per chunk on one warp
        // against 190-380 cycles of tensor work, and that warp paced the whole chain.  The MMAs of chunk 0 overwrite the
        // accumulator: the second warp starts a GEMM only after they have COMPLETED (bar_first, committed by this warp).
        const uint32_t mw = uni(warp == 1 ? 0u : 1u);
        uint32_t wi = 0, rc = 0, par0 = 0u, par1 = 0u; // parities of the chunk barriers, one bit per chunk slot and region
        uint32_t nd = 0, nf = 0;                       // phases of bar_drained / bar_first consumed so far
        bool pending_drain = false;                    // the last accumulator written has not been waited for yet
        for (int t = tu_beg; t < tu_end; ++t) {
            const int gi = (int)uni((uint32_t)find_group(gsm, n_gc, t));
            const FusedGroup &g = gsm[gi];
            const int n_stages = (int)uni((uint32_t)g.n_stages);
            for (int j = 0; j < n_stages; ++j) {
                const int K = (int)uni((uint32_t)g.st[j].K), Np = (int)uni((uint32_t)g.st[j].N);
                const int n_total = (WIDE && j + 1 == n_stages) ? (int)uni((uint32_t)g.st[j].n_total) : Np;
                const uint32_t ra = (rc + (uint32_t)j) & 1u, rd = ra ^ 1u;
                const uint32_t a_base = tb + ra * REGION_COLS, acc = tb + rd * REGION_COLS;
                const int nch_tot = K / CH, nkb = (K + KBH - 1) / KBH;
                // passes: only the last GEMM of a wide chain has more than one (its n_total output columns, Np at a time, from
                // the same operand into the same region, which the epilogue must have drained in between)
                int col = 0;
                do { // (one pass, statically, in the narrow kernels)
                    const int N = WIDE && n_total - col < Np ? n_total - col : Np;
                    const bool wide = N > 128; // two MMAs per product term: columns [0, 128) and [128, N)
                    const uint32_t rows0 = (uint32_t)part_rows(N, 0), rows1 = wide ? (uint32_t)part_rows(N, 1) : 8u;
                    const uint32_t idesc0 = (1u << 4) | ((rows0 >> 3) << 17) | ((uint32_t)(TILE_M >> 4) << 24);
                    const uint32_t idesc1 = (1u << 4) | ((rows1 >> 3) << 17) | ((uint32_t)(TILE_M >> 4) << 24);
                    // the first GEMM of a tile, and every further pass of the last one, write a region whose previous
                    // accumulator (last GEMM of the previous tile / previous pass) the epilogue must have read
                    if (pending_drain && (j == 0 || col > 0)) {
                        mbar_wait(bar_drained, nd & 1u, 200, t - tu_beg);
                        ++nd;
                        pending_drain = false;
                        tc_fence_after();
                    }
                    bool first_pending = mw != 0u; // (second warp) chunk 0 of this GEMM / pass not known to be complete yet
                    for (int kb = 0; kb < nkb; ++kb) {
                        const uint32_t e0 = wi % NW, e1 = (wi + 1) % NW;
                        mbar_wait(bar_wfull + 8 * e0, (wi / NW) & 1, 220 + j, (t - tu_beg) * 100 + kb);
                        if (wide) mbar_wait(bar_wfull + 8 * e1, ((wi + 1) / NW) & 1, 230 + j, (t - tu_beg) * 100 + kb);
                        const uint32_t b0 = wr + e0 * W_ENTRY_BYTES, b1 = wr + e1 * W_ENTRY_BYTES;
                        const uint64_t d0hi = make_kmajor_sw128_desc(b0), d0lo = make_kmajor_sw128_desc(b0 + rows0 * 128u);
                        const uint64_t d1hi = make_kmajor_sw128_desc(b1), d1lo = make_kmajor_sw128_desc(b1 + rows1 * 128u);
                        const int nh = nch_tot - 4 * kb < 4 ? nch_tot - 4 * kb : 4;
                        // one wait and one election per chunk (measured against the chunks of a K block in one batch, or the
                        // first alone and the other three together: 0.203 against 0.214 ms for the narrow chain; batching only
                        // the first / last GEMM of a wide chain: config 5 7.35 -> 7.83 ms)
                        for (int h = 0; h < nh; ++h) {
                            const int c = 4 * kb + h, slot = WIDE ? c % MAX_CHUNKS : c; // an operand wider than a region reuses its slots
                            if ((uint32_t)(h & 1) != mw) continue;
                            if (!WIDE || col == 0) { // (further passes multiply the operand that is already there)
                                mbar_wait(bar_ready + 8 * (ra * MAX_CHUNKS + slot), ((ra ? par1 : par0) >> slot) & 1u, 240 + j, (t - tu_beg) * 100 + c);
                                if (ra) par1 ^= 1u << slot; else par0 ^= 1u << slot;
                                tc_fence_after();
                            }
                            if (first_pending) {
                                mbar_wait(bar_first, nf & 1u, 250 + j, (t - tu_beg) * 100 + c);
                                ++nf;
                                first_pending = false;
                                tc_fence_after();
                            }
                            if (elect_one()) {
                                const uint32_t a_hi = a_base + (uint32_t)(CH * slot), a_lo = a_hi + 8;
                                const uint64_t koff = (uint64_t)(2 * h); // 16 fp16 = 32 B along the swizzled row
                                mma_f16_ts(acc, a_lo, d0hi + koff, idesc0, c ? 1u : 0u);
                                mma_f16_ts(acc, a_hi, d0lo + koff, idesc0, 1u);
                                mma_f16_ts(acc, a_hi, d0hi + koff, idesc0, 1u);
                                if (wide) {
                                    mma_f16_ts(acc + 128, a_lo, d1hi + koff, idesc1, c ? 1u : 0u);
                                    mma_f16_ts(acc + 128, a_hi, d1lo + koff, idesc1, 1u);
                                    mma_f16_ts(acc + 128, a_hi, d1hi + koff, idesc1, 1u);
                                }
                                if (c == 0) tc_commit(bar_first);
                                // (each warp after its last slot of a pass of 16: the slots may be rewritten)
                                if (WIDE && slot >= MAX_CHUNKS - 2 && (c | (MAX_CHUNKS - 1)) + 1 < nch_tot) tc_commit(bar_pass);
                                if (h + 2 >= nh) { // this warp's last chunk of the K block
                                    tc_commit(bar_wempty + 8 * e0);
                                    if (wide) tc_commit(bar_wempty + 8 * e1);
                                    if (kb + 1 == nkb) tc_commit(bar_accf + 8 * rd);
                                }
                            }
                            __syncwarp();
                        }
                        if ((uint32_t)nh <= mw) { // no chunk of this K block was this warp's: it releases the weights all the same
                            if (elect_one()) {
                                tc_commit(bar_wempty + 8 * e0);
                                if (wide) tc_commit(bar_wempty + 8 * e1);
                                if (kb + 1 == nkb) tc_commit(bar_accf + 8 * rd);
                            }
                            __syncwarp();
                        }
                        wi += wide ? 2u : 1u;
                    }
                    if (first_pending) { // (a GEMM of a single chunk: the phase is taken all the same)
                        mbar_wait(bar_first, nf & 1u, 260 + j, t - tu_beg);
                        ++nf;
                    }
                    if (j + 1 == n_stages) pending_drain = true;
                } while (WIDE && (col += Np) < n_total);
            }
            rc += (uint32_t)n_stages + 1u;
        }
    } else {
        // ===== epilogue: warps 2..17; warp -> TMEM lane quarter warp & 3; set s = (warp - 2) / 4 takes the 16-column chunks
        // s, s + 4, ... of an accumulator (and of the chain's input).  Lane l owns row quarter * 32 + l of the tile.
        const int ew = warp - 2;
        const int quarter = warp & 3;
        const int set = ew >> 2;
        const int row = quarter * 32 + lane;
        const uint32_t lane_addr = tmem_base + ((uint32_t)(quarter * 32) << 16);
        const uint32_t stg = stg_base + (uint32_t)ew * EPI_STG_BYTES;
        uint32_t rc = 0, use0 = 0u, use1 = 0u, a_ph = 0, pass_cnt = 0; // a_ph: phases of this set's input-ring entry taken so far
        int cur_gi = -1;
        float vmax = 0.f;
        for (int t = t_beg; t < t_end; ++t) {
            const int gi = find_group(gsm, n_gc, t);
            const FusedGroup &g = gsm[gi];
            if (gi != cur_gi) {
                // biases (x 16) of the forward GEMMs and w4 of this group -> shared memory (a chunk reads them as broadcasts)
                asm volatile("bar.sync 1, %0;" ::"n"(EPI_WARPS * 32) : "memory"); // nobody still reads the previous group's
                float *sbp = reinterpret_cast<float *>(smem_raw + (sb_base - smem_u32(smem_raw)));
                const int et = (int)threadIdx.x - 64;
                for (int j = 0; j < g.n_stages; ++j)
                    if (g.st[j].epi == FE_FWD || g.st[j].epi == FE_OUT)
                        for (int k = et; k < g.st[j].N; k += EPI_WARPS * 32) sbp[g.st[j].brow * REGION_COLS + k] = g.st[j].bias[k];
                for (int k = et; k < g.h3; k += EPI_WARPS * 32) sbp[3 * REGION_COLS + k] = g.w4[k];
                asm volatile("bar.sync 1, %0;" ::"n"(EPI_WARPS * 32) : "memory");
                cur_gi = gi;
            }
            const int m0 = (t - g.tile0) * TILE_M;
            const int mrow0 = m0 + quarter * 32;
            const int m = mrow0 + lane;
            const bool rowok = m < g.M;
            {
                // chain input (fp32 rows through the TMA ring) -> fp16 hi / lo chunks.  Their region was the operand of the
                // previous tile's last GEMM, which this warp has seen complete (accumulator barrier of that GEMM).
                const int nch0 = g.st[0].K / CH;
                const uint32_t r0 = rc & 1u;
                for (int c_pass = 0, pass = 0; c_pass < (WIDE ? nch0 : 1); c_pass += MAX_CHUNKS, ++pass) {
                    // an input wider than a region goes through it in passes of 16 chunks: a slot is written again once the
                    // MMAs of the pass before have completed (bar_pass, committed by both MMA warps per pass).  Every warp
                    // takes every phase of this barrier, with or without a chunk in the pass: an mbarrier wait names a
                    // phase by its parity only, so a waiter that skipped one would take the phase before for its own.
                    if (WIDE && pass > 0) {
                        mbar_wait(bar_pass, (pass_cnt + (uint32_t)pass - 1u) & 1u, 330, (t - t_beg) * 100 + pass);
                        tc_fence_after();
                    }
                    const int c_end = c_pass + MAX_CHUNKS < nch0 ? c_pass + MAX_CHUNKS : nch0;
                    for (int c = c_pass + set; c < c_end; c += EPI_SETS) {
                        const uint32_t e = (uint32_t)(set >> 1); // ring entry of this set's input tiles (producer: tile k -> k & 1)
                        mbar_wait(bar_afull + 8 * e, a_ph & 1u, 300, (t - t_beg) * 100 + c);
                        ++a_ph;
                        const uint32_t arow = a_ring + e * A_TILE_BYTES + row * 128;
                        float x[16];
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            const uint32_t addr = arow + (uint32_t)(((4 * (c & 1) + q) ^ (row & 7)) << 4);
                            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(x[4 * q]), "=f"(x[4 * q + 1]), "=f"(x[4 * q + 2]), "=f"(x[4 * q + 3]) : "r"(addr));
                        }
                        uint32_t v[16];
#pragma unroll
                        for (int q = 0; q < 16; ++q) { x[q] *= ACT_SCALE; vmax = fmaxf(vmax, fabsf(x[q])); }
                        split16(x, v);
                        __syncwarp();
                        if (lane == 0) mbar_arrive(bar_aempty + 8 * e); // this warp's half of the tile is in registers
                        tmem_st16(lane_addr + r0 * REGION_COLS + (uint32_t)(CH * (WIDE ? c % MAX_CHUNKS : c)), v);
                        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(bar_ready + 8 * (r0 * MAX_CHUNKS + (WIDE ? c % MAX_CHUNKS : c)));
                    }
                }
                if (WIDE) pass_cnt += (uint32_t)((nch0 - 1) / MAX_CHUNKS);
            }
            const int lane_set = lane | (set << 8), aux = t - t_beg;
#define NNP_FUSED_PASS(J, COL, NCOLS)                                                                                         \
    {                                                                                                                         \
        const uint32_t accf = (bar_accf + 8 * rd) | (((rd ? use1 : use0) & 1u) << 31);                                        \
        if (rd) ++use1; else ++use0;                                                                                          \
        const float2 r = epi_stage<chain_epi(CHAIN, J)>(&g, J, mrow0, lane_set, lane_addr + rd * REGION_COLS, stg, accf,      \
                                                        bar_ready + 8 * (rd * MAX_CHUNKS), sb_base, alpha, aux, NCOLS, COL);  \
        vmax = fmaxf(vmax, r.x);                                                                                              \
        if (chain_epi(CHAIN, J) == FE_OUT && rowok) atomicAdd(g.e_atom + m, r.y * (1.0f / ACT_SCALE));                        \
        if (J + 1 == chain_len(CHAIN)) { /* this accumulator has left tensor memory (for this warp): the next pass / tile    \
                                            may overwrite it */                                                              \
            tc_fence_before();                                                                                                \
            __syncwarp();                                                                                                     \
            if (lane == 0) mbar_arrive(bar_drained);                                                                          \
        }                                                                                                                     \
    }
#define NNP_FUSED_STAGE(J)                                                                                                    \
    if (J < chain_len(CHAIN)) {                                                                                               \
        const uint32_t rd = (rc + (uint32_t)J + 1u) & 1u;                                                                     \
        if (WIDE && J + 1 == chain_len(CHAIN)) { /* the last GEMM of a wide chain: passes of N of its n_total columns */      \
            const int n_pass_cols = g.st[J].N, n_total = g.st[J].n_total;                                                     \
            for (int col = 0; col < n_total; col += n_pass_cols)                                                              \
                NNP_FUSED_PASS(J, col, n_total - col < n_pass_cols ? n_total - col : n_pass_cols)                             \
        } else {                                                                                                              \
            NNP_FUSED_PASS(J, 0, g.st[J].N)                                                                                   \
        }                                                                                                                     \
    }
            NNP_FUSED_STAGE(0) NNP_FUSED_STAGE(1) NNP_FUSED_STAGE(2) NNP_FUSED_STAGE(3) NNP_FUSED_STAGE(4) NNP_FUSED_STAGE(5)
#undef NNP_FUSED_STAGE
#undef NNP_FUSED_PASS
            rc += (uint32_t)g.n_stages + 1u;
        }
        if (vmax > RANGE_LIMIT) atomicOr(&flags[0], NNP_FLAG_RANGE);
    }
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
    }
}

// Packs one weight matrix Bt [N][K] (K contiguous; the B operand of D = A . Bt^T), multiplied by `scale`, into the tile
// images the kernel copies with one bulk load each: for every K block of 64 and part p (rows [0,128) / [128,N)): the
// fp16-hi tile then the fp16-lo tile, rows of 128 B (zero beyond K), 16-byte chunk c of row r stored at chunk position
// c ^ (r & 7) (128-byte swizzle).
__global__ void k_pack_weights(const float *__restrict__ Bt, int N, int K, int ldb, float scale, uint8_t *__restrict__ dst)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x; // one 16-byte chunk (8 fp16) of one row of one K block
    const int nkb = (K + KBH - 1) / KBH;
    if (idx >= N * nkb * 8) return;
    const int c = idx & 7, n = (idx >> 3) % N, kb = (idx >> 3) / N;
    const int p = n >= 128 ? 1 : 0, rows = p == 0 ? (N > 128 ? 128 : N) : N - 128, r = n - 128 * p;
    // K block kb: [part 0: hi rows0 x 128 | lo rows0 x 128][part 1: hi | lo]
    const size_t kb_bytes = (size_t)2 * N * 128;
    uint8_t *tile = dst + kb * kb_bytes + (p ? (size_t)2 * (N > 128 ? 128 : N) * 128 : 0);
    uint32_t hi[4], lo[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int k = kb * KBH + 8 * c + 2 * q;
        const float x0 = k < K ? Bt[(size_t)n * ldb + k] * scale : 0.f;
        const float x1 = k + 1 < K ? Bt[(size_t)n * ldb + k + 1] * scale : 0.f;
        const __half2 h = __floats2half2_rn(x0, x1);
        const float2 hf = __half22float2(h);
        const __half2 l = __floats2half2_rn(x0 - hf.x, x1 - hf.y);
        hi[q] = *reinterpret_cast<const uint32_t *>(&h);
        lo[q] = *reinterpret_cast<const uint32_t *>(&l);
    }
    const size_t off = (size_t)r * 128 + (size_t)((c ^ (r & 7)) << 4);
    *reinterpret_cast<uint4 *>(tile + off) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4 *>(tile + (size_t)rows * 128 + off) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
}

__global__ void k_scale_copy(const float *__restrict__ src, int n, float scale, float *__restrict__ dst)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src[i] * scale;
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
    cuuint32_t box[2] = {(cuuint32_t)KBF, (cuuint32_t)TILE_M};
    cuuint32_t estr[2] = {1, 1};
    return g_encode(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void *)base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// bytes of the packed tiles of one matrix Bt [N][K]
size_t packed_bytes(int N, int K) { return (size_t)((K + KBH - 1) / KBH) * 2 * N * 128; }

// power-of-two weight scale: max |w| 2^e in [2^13, 2^14)
int weight_shift(float wmax)
{
    if (!(wmax > 0.f) || !isfinite(wmax)) return 0;
    int e;
    frexpf(wmax, &e); // wmax = f 2^e, f in [0.5, 1)
    int sh = 14 - e;
    if (sh > 40) sh = 40;
    if (sh < -40) sh = -40;
    return sh;
}

} // namespace

struct nnp_fused {
    int kind;                    // 0: not usable for the loaded system (the six-launch path runs), 1: the fused chain
    int n_groups, n_tiles, grid;
    FusedGroup *d_groups;        // [n_nets * S]
    int *d_cta_tiles;            // [grid + 1]
    uint8_t *d_wblob;            // packed weights of every (network, species): sized at first use for the largest layout
    float *d_bias16;             // [n_nets * S][3][256] biases * 2^ACT_SHIFT
    size_t wblob_bytes;
    size_t w_off[64][MAX_STAGES + 1]; // per (network, species): byte offsets of F1 F2 F3 B3 B2 B1 in the blob
    unsigned packed_mask;        // species mask the layer-1 tiles were packed for (0: nothing packed yet)
    int last_off[NNP_MAX_SPECIES + 1], last_kpad; // bucket offsets / G pitch the tables were built for (last_kpad = 0: none)
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
    fr(c, f->d_groups); fr(c, f->d_cta_tiles); fr(c, f->d_wblob); fr(c, f->d_bias16);
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
// (c->fused->kind = 0: the six-launch 3xTF32 path runs).
int nnp_fused_setup(nnp_ctx *c)
{
    if (c->mm_mode != NNP_MM_3XF16_TC || c->no_fused) return NNP_OK;
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
    const int kpad = c->aev.kpad;
    // same species counts and layout as the last system (e.g. one structure evaluated again and again through
    // nnp_energy_forces_host): the packed weights, the group table and the tile ranges stand as they are
    if (f->kind == 1 && f->last_kpad == kpad && f->packed_mask == c->present_mask &&
        memcmp(f->last_off, c->bucket_off, sizeof(f->last_off)) == 0)
        return NNP_OK;
    f->kind = 0;
    f->last_kpad = 0;
    // widths a 256-column region holds; every accumulator must give all four epilogue sets a chunk
    for (int s = 0; s < S; ++s)
        for (int l = 1; l <= 3; ++l)
            if (c->widths[s][l] > REGION_COLS || c->widths[s][l] < EPI_SETS * CH) return NNP_OK;
    const size_t k0max = c->kpad_full;
    // ---- packed weights: per (net, species) the six matrices in chain order; sized for the largest layout once
    if (!f->d_wblob) {
        size_t tot = 0;
        for (int net = 0; net < nn; ++net)
            for (int s = 0; s < S; ++s) {
                const int h1 = c->widths[s][1], h2 = c->widths[s][2], h3 = c->widths[s][3];
                tot += packed_bytes(h1, (int)k0max) + packed_bytes((int)k0max, h1) + packed_bytes(h2, h1) + packed_bytes(h1, h2) +
                       packed_bytes(h3, h2) + packed_bytes(h2, h3);
            }
        f->d_wblob = (uint8_t *)fused_alloc(c, tot);
        if (!f->d_wblob) { c->err = "fused MLP: weight tile allocation failed"; return NNP_ENOMEM; }
        f->wblob_bytes = tot;
        f->d_groups = (FusedGroup *)fused_alloc(c, sizeof(FusedGroup) * 64);
        f->d_cta_tiles = (int *)fused_alloc(c, sizeof(int) * (f->num_sms + 1));
        f->d_bias16 = (float *)fused_alloc(c, sizeof(float) * (size_t)nn * S * 3 * REGION_COLS);
        if (!f->d_groups || !f->d_cta_tiles || !f->d_bias16) { c->err = "fused MLP: table allocation failed"; return NNP_ENOMEM; }
        f->packed_mask = 0;
    }
    auto pack = [&](const float *Bt, int N, int K, int ldb, int shift, uint8_t *dst) {
        const int total = N * ((K + KBH - 1) / KBH) * 8;
        k_pack_weights<<<nnp_div_up(total, 256), 256, 0, c->stream>>>(Bt, N, K, ldb, ldexpf(1.0f, shift), dst);
        c->launches += 1;
    };
    const bool repack_l1 = f->packed_mask != c->present_mask;
    const bool first_pack = f->packed_mask == 0;
    int wsh[64][3]; // weight shifts of layers 1..3 per (network, species)
    {
        size_t o = 0;
        for (int net = 0; net < nn; ++net)
            for (int s = 0; s < S; ++s) {
                const int q = net * S + s;
                const int h1 = c->widths[s][1], h2 = c->widths[s][2], h3 = c->widths[s][3];
                const LayerW *L = &c->layers[((size_t)net * S + s) * NNP_NLAYERS];
                const Layer1C &l1 = c->l1c[(size_t)net * S + s];
                for (int l = 0; l < 3; ++l) wsh[q][l] = weight_shift(L[l].wmax);
                // F1: B = W1^T [h1][kpad]; F2: W2^T [h2][h1]; F3: W3^T [h3][h2]; B3: W3 [h2][h3]; B2: W2 [h1][h2]; B1: W1 [kpad][h1]
                f->w_off[q][0] = o; o += packed_bytes(h1, (int)k0max);
                f->w_off[q][1] = o; o += packed_bytes(h2, h1);
                f->w_off[q][2] = o; o += packed_bytes(h3, h2);
                f->w_off[q][3] = o; o += packed_bytes(h2, h3);
                f->w_off[q][4] = o; o += packed_bytes(h1, h2);
                f->w_off[q][5] = o; o += packed_bytes((int)k0max, h1);
                f->w_off[q][6] = o;
                if (first_pack) {
                    pack(L[1].Wt, h2, h1, h1, wsh[q][1], f->d_wblob + f->w_off[q][1]);
                    pack(L[2].Wt, h3, h2, h2, wsh[q][2], f->d_wblob + f->w_off[q][2]);
                    pack(L[2].W, h2, h3, h3, wsh[q][2], f->d_wblob + f->w_off[q][3]);
                    pack(L[1].W, h1, h2, h2, wsh[q][1], f->d_wblob + f->w_off[q][4]);
                    for (int l = 0; l < 3; ++l) {
                        k_scale_copy<<<1, 256, 0, c->stream>>>(L[l].b, c->widths[s][l + 1], ACT_SCALE, f->d_bias16 + ((size_t)q * 3 + l) * REGION_COLS);
                        c->launches += 1;
                    }
                }
                if (repack_l1) {
                    pack(l1.Wt, h1, kpad, kpad, wsh[q][0], f->d_wblob + f->w_off[q][0]);
                    size_t ob = f->w_off[q][5]; // dE/dG: passes of <= 256 output columns, packed one after the other
                    for (int col = 0; col < kpad; col += REGION_COLS) {
                        const int nq = kpad - col < REGION_COLS ? kpad - col : REGION_COLS;
                        pack(l1.W + (size_t)col * h1, nq, h1, h1, wsh[q][0], f->d_wblob + ob);
                        ob += packed_bytes(nq, h1);
                    }
                }
            }
    }
    f->packed_mask = c->present_mask;

    // ---- groups (one per network and species present) and tiles
    std::vector<FusedGroup> groups;
    std::vector<long long> cost;
    int tiles = 0;
    const float alpha = c->alpha;
    for (int net = 0; net < nn; ++net)
        for (int s = 0; s < S; ++s) {
            const int off = c->bucket_off[s], M = c->bucket_off[s + 1] - off;
            if (M == 0) continue;
            const int q = net * S + s;
            const int h1 = c->widths[s][1], h2 = c->widths[s][2], h3 = c->widths[s][3];
            const LayerW *L = &c->layers[((size_t)net * S + s) * NNP_NLAYERS];
            float *H0 = c->H[0] + ((size_t)net * c->max_atoms + off) * c->hmax[0];
            float *H1 = c->H[1] + ((size_t)net * c->max_atoms + off) * c->hmax[1];
            const float *b16 = f->d_bias16 + (size_t)q * 3 * REGION_COLS;
            FusedGroup g;
            memset(&g, 0, sizeof(g));
            g.wblob = f->d_wblob;
            g.w4 = L[3].W;
            g.e_atom = c->e_atom + off;
            g.M = M;
            g.h3 = h3;
            g.tile0 = tiles;
            g.n_tiles = nnp_div_up(M, TILE_M);
            // acc = sum (16 a)(2^sh w): forward epilogues want 16 z = acc 2^-sh; reverse operand-producing epilogues
            // 16 delta = acc 2^-sh celu'(h) with the stash holding 16 h; output epilogues the true value acc 2^-(sh + 4)
            auto fwd = [&](int j, int K, int N, int epi, size_t w_off, const float *bias, float *stash, int ld, int sh, int brow) {
                FusedStage &st = g.st[j];
                st.K = K; st.N = N; st.epi = epi; st.w_off = (uint32_t)w_off; st.bias = bias; st.stash = stash; st.ld_stash = ld;
                st.c_acc = ldexpf(1.0f, -sh);
                st.brow = brow;
                st.n_total = N;
            };
            auto bwd = [&](int j, int K, int N, int epi, size_t w_off, float *stash, int ld, int sh) {
                FusedStage &st = g.st[j];
                st.K = K; st.N = N < REGION_COLS ? N : REGION_COLS; st.n_total = N; st.epi = epi; st.w_off = (uint32_t)w_off; st.stash = stash; st.ld_stash = ld;
                const float s2 = ldexpf(1.0f, -sh);
                if (epi == FE_BWD) { st.gs = s2 / (alpha * ACT_SCALE); st.gc = s2; }                       // stash = 16 h, out = 16 delta
                st.c_acc = s2 / ACT_SCALE;                                                                  // FE_ST / FE_RED
            };
            if (f->w_off[q][6] > 0xffffffffull) { c->err = "fused MLP: weight blob exceeds 4 GiB"; return NNP_EINVAL; }
            g.n_stages = 6;
            if (!make_map_a(&g.mapA, c->G + (size_t)off * kpad, M, kpad, kpad)) { c->err = "cuTensorMapEncodeTiled failed"; return NNP_ECUDA; }
            fwd(0, kpad, h1, FE_FWD, f->w_off[q][0], b16, H0, c->hmax[0], wsh[q][0], 0);
            fwd(1, h1, h2, FE_FWD, f->w_off[q][1], b16 + REGION_COLS, H1, c->hmax[1], wsh[q][1], 1);
            fwd(2, h2, h3, FE_OUT, f->w_off[q][2], b16 + 2 * REGION_COLS, nullptr, 0, wsh[q][2], 2);
            bwd(3, h3, h2, FE_BWD, f->w_off[q][3], H1, c->hmax[1], wsh[q][2]);
            bwd(4, h2, h1, FE_BWD, f->w_off[q][4], H0, c->hmax[0], wsh[q][1]);
            bwd(5, h1, kpad, nn > 1 ? FE_RED : FE_ST, f->w_off[q][5], nullptr, 0, wsh[q][0]);
            g.out = c->dG + (size_t)off * kpad;
            g.ldo = kpad;
            // Cost of a tile in cycles, for the split of the tiles over the CTAs.  Measured per CTA (clock64 around the tile
            // loop, 98k-atom water box): a tile takes 3.1 k cycles per round of the epilogue (the sixteen warps drain 64
            // accumulator columns per round) - 59.0 k for the H network (19 rounds), 49.7 k for O (16 rounds); a GEMM whose
            // MMAs take longer than its rounds (the first of a wide chain) counts with those, and the conversion of the chain's
            // input with 2 k cycles per 64 columns.  (The first model, MMA cycles + a constant per GEMM, made O tiles 0.78 of an
            // H tile: CTAs with seven O tiles ran 349 k cycles against a mean of 290 k.)
            long long cst = 2000LL * ((g.st[0].K + 63) / 64);
            for (int j = 0; j < g.n_stages; ++j) {
                const long long rounds = 3100LL * ((g.st[j].n_total + 63) / 64), mma = (long long)(g.st[j].K / CH) * 3 * (g.st[j].n_total / 2);
                cst += rounds > mma ? rounds : mma;
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
    f->grid = grid;
    for (int b = 0; b < grid; ++b) { // the kernel keeps the descriptors of a CTA's groups in shared memory
        int span = 0;
        for (size_t q = 0; q < groups.size(); ++q)
            if (groups[q].tile0 < cta[b + 1] && groups[q].tile0 + groups[q].n_tiles > cta[b]) ++span;
        if (span > GCACHE) return NNP_OK; // kind stays 0: the six-launch path
    }
    if (cudaMemcpyAsync(f->d_groups, groups.data(), sizeof(FusedGroup) * groups.size(), cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaMemcpyAsync(f->d_cta_tiles, cta.data(), sizeof(int) * (grid + 1), cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess) { // the host vectors go out of scope
        c->err = std::string("fused MLP: table upload failed: ") + cudaGetErrorString(cudaGetLastError());
        return NNP_ECUDA;
    }
    f->kind = 1;
    f->last_kpad = kpad;
    memcpy(f->last_off, c->bucket_off, sizeof(f->last_off));
    return NNP_OK;
}

int nnp_fused_kind(const nnp_ctx *c) { return c->fused ? c->fused->kind : 0; }

// Enqueues the fused chain (all six GEMMs of every network and species in one launch).
void nnp_launch_mlp_fused(nnp_ctx *c)
{
    nnp_fused *f = c->fused;
    typedef void (*Kern)(const FusedGroup *, int, const int *, float, int *);
    static const Kern kerns[4] = {k_mlp_fused<CHAIN_FULL, false>, k_mlp_fused<CHAIN_FULL_RED, false>, k_mlp_fused<CHAIN_FULL, true>,
                                  k_mlp_fused<CHAIN_FULL_RED, true>};
    static bool attr_set = false;
    if (!attr_set) {
        for (int k = 0; k < 4; ++k) cudaFuncSetAttribute(kerns[k], cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        attr_set = true;
    }
    const Kern kern = kerns[(c->n_nets > 1 ? 1 : 0) + (c->aev.kpad > REGION_COLS ? 2 : 0)];
    kern<<<f->grid, THREADS, SMEM_BYTES, c->stream>>>(f->d_groups, f->n_groups, f->d_cta_tiles, c->alpha, c->flags);
    c->launches += 1;
}
