// Stage 3/4, mm_mode = NNP_MM_FP32_SIMT / NNP_MM_FP64_SIMT: species-grouped GEMMs on the CUDA cores with the layer
// epilogues fused (bias + CELU; last hidden layer folded with the 1-wide output layer and CELU'; reverse-mode
// delta chain with CELU').  ChemicalNet; "highest" fp32 precision, L315-321.
// ACC = float: the full-fp32 path on the device.  ACC = double: the fp64 leg of the precision study (Fig. 3
// compares bf16 / TF32 / fp32 / fp64 matmuls): fp32 operands, every product and sum of the contraction, the bias, CELU and
// CELU' in fp64 (DFMA), the result rounded once to the fp32 activation buffers.  The tensor-core path is mlp_tc.cu.
#include "nnp_internal.cuh"

namespace {

constexpr int BM = 128, BN = 64, BK = 16, THREADS = 256;
constexpr int TM = 8, TN = 4; // per-thread micro-tile: 16 x 16 threads

// Branch-free CELU: max(x,0) + alpha (2^(min(x,0) log2e / alpha) - 1).  (A conditional form makes the compiler
// emit one divergent branch per element, which serialised the tensor-core epilogue.)
__device__ __forceinline__ float celu_fwd(float x, float alpha, float inv_alpha)
{
    float e;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(fminf(x, 0.f) * (inv_alpha * 1.4426950408889634f)));
    return fmaxf(x, 0.f) + alpha * (e - 1.0f);
}
// CELU'(z) expressed with h = CELU(z): 1 for h > 0, else exp(z/alpha) = 1 + h/alpha
__device__ __forceinline__ float celu_grad_from_h(float h, float inv_alpha) { return fmaf(fminf(h, 0.f), inv_alpha, 1.0f); }

__device__ __forceinline__ double celu_fwd(double x, double alpha, double inv_alpha)
{
    return fmax(x, 0.0) + alpha * expm1(fmin(x, 0.0) * inv_alpha);
}
__device__ __forceinline__ double celu_grad_from_h(double h, double inv_alpha) { return fma(fmin(h, 0.0), inv_alpha, 1.0); }

template <int EPI, typename ACC>
__global__ void __launch_bounds__(THREADS)
k_gemm_simt(GemmBatch batch)
{
    __shared__ __align__(16) float As[2][BK][BM + 4];
    __shared__ __align__(16) float Bs[2][BK][BN];

    // tile -> (group, m-tile)
    int gi = 0;
    while (gi + 1 < batch.n_groups && (int)blockIdx.x >= batch.tile_off[gi + 1]) ++gi;
    const GemmGroup &g = batch.g[gi];
    const int m0 = ((int)blockIdx.x - batch.tile_off[gi]) * BM;
    const int n0 = blockIdx.y * BN;
    if (n0 >= g.N) return;

    const int tid = threadIdx.x;
    const int ty = tid / 16, tx = tid % 16;
    // A loader: 128 rows x 16 k = 512 float4, two per thread; B loader: 16 k x 64 n = 256 float4, one per thread
    const int a_row = tid / 4, a_k4 = (tid % 4) * 4;
    const int b_k = tid / 16, b_n4 = (tid % 16) * 4;

    ACC acc[TM][TN];
#pragma unroll
    for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) acc[i][j] = (ACC)0;

    float4 ra[2], rb;
    auto gload = [&](int k0) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int row = m0 + a_row + h * 64;
            ra[h] = row < g.M ? *reinterpret_cast<const float4 *>(g.A + (size_t)row * g.lda + k0 + a_k4)
                              : make_float4(0.f, 0.f, 0.f, 0.f);
        }
        const int col = n0 + b_n4;
        rb = col < g.N ? *reinterpret_cast<const float4 *>(g.B + (size_t)(k0 + b_k) * g.N + col)
                       : make_float4(0.f, 0.f, 0.f, 0.f);
    };
    auto sstore = [&](int buf) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int r = a_row + h * 64;
            As[buf][a_k4 + 0][r] = ra[h].x;
            As[buf][a_k4 + 1][r] = ra[h].y;
            As[buf][a_k4 + 2][r] = ra[h].z;
            As[buf][a_k4 + 3][r] = ra[h].w;
        }
        *reinterpret_cast<float4 *>(&Bs[buf][b_k][b_n4]) = rb;
    };

    gload(0);
    sstore(0);
    __syncthreads();
    const int nk = g.K / BK;
    for (int kt = 0; kt < nk; ++kt) {
        const int buf = kt & 1;
        if (kt + 1 < nk) gload((kt + 1) * BK);
#pragma unroll
        for (int k = 0; k < BK; ++k) {
            const float4 a0 = *reinterpret_cast<const float4 *>(&As[buf][k][ty * TM]);
            const float4 a1 = *reinterpret_cast<const float4 *>(&As[buf][k][ty * TM + 4]);
            const float4 b = *reinterpret_cast<const float4 *>(&Bs[buf][k][tx * TN]);
            const float av[TM] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
            const float bv[TN] = {b.x, b.y, b.z, b.w};
#pragma unroll
            for (int i = 0; i < TM; ++i)
#pragma unroll
                for (int j = 0; j < TN; ++j) acc[i][j] = fma((ACC)av[i], (ACC)bv[j], acc[i][j]);
        }
        if (kt + 1 < nk) {
            sstore(buf ^ 1);
            __syncthreads();
        }
    }

    // ---- epilogue
    const ACC alpha = (ACC)batch.alpha, inv_alpha = (ACC)1 / (ACC)batch.alpha;
    const int col = n0 + tx * TN;
    const bool colok = col < g.N; // N is a multiple of 32 and TN = 4: a thread's 4 columns are all in or all out
    float bias[TN] = {0.f, 0.f, 0.f, 0.f}, w4[TN] = {0.f, 0.f, 0.f, 0.f};
    if (colok && (EPI == EPI_CELU || EPI == EPI_CELU_OUT)) {
        const float4 b4 = *reinterpret_cast<const float4 *>(g.bias + col);
        bias[0] = b4.x; bias[1] = b4.y; bias[2] = b4.z; bias[3] = b4.w;
    }
    if (colok && EPI == EPI_CELU_OUT) {
        const float4 w = *reinterpret_cast<const float4 *>(g.w4 + col);
        w4[0] = w.x; w4[1] = w.y; w4[2] = w.z; w4[3] = w.w;
    }
#pragma unroll
    for (int i = 0; i < TM; ++i) {
        const int row = m0 + ty * TM + i;
        ACC esum = (ACC)0;
        float4 out;
        float *o = reinterpret_cast<float *>(&out);
        float4 prev = make_float4(0.f, 0.f, 0.f, 0.f);
        float *cp = g.C + (size_t)row * g.ldc + col;
        if (row < g.M && colok && (EPI == EPI_DCELU || EPI == EPI_ACCUM)) prev = *reinterpret_cast<const float4 *>(cp);
        const float *pv = reinterpret_cast<const float *>(&prev);
#pragma unroll
        for (int j = 0; j < TN; ++j) {
            ACC v = acc[i][j];
            if (EPI == EPI_CELU) v = celu_fwd(v + (ACC)bias[j], alpha, inv_alpha);
            if (EPI == EPI_CELU_OUT) {
                const ACC h = celu_fwd(v + (ACC)bias[j], alpha, inv_alpha);
                esum = fma(h, (ACC)w4[j], esum);
                v = (ACC)w4[j] * celu_grad_from_h(h, inv_alpha);
            }
            if (EPI == EPI_DCELU) v *= celu_grad_from_h((ACC)pv[j], inv_alpha);
            if (EPI == EPI_ACCUM) v += (ACC)pv[j];
            o[j] = (float)v;
        }
        if (EPI == EPI_CELU_OUT) {
            // reduce the partial dot product over the 16 threads (tx) that share this row
#pragma unroll
            for (int off = 8; off >= 1; off >>= 1) esum += __shfl_xor_sync(0xffffffffu, esum, off);
            if (tx == 0 && row < g.M) atomicAdd(g.e_atom + row, (float)esum);
        }
        if (row < g.M && colok) *reinterpret_cast<float4 *>(cp) = out;
    }
}

} // namespace

template <typename ACC>
static void launch_simt(cudaStream_t st, const GemmBatch &b, int epi, dim3 grid)
{
    switch (epi) {
    case EPI_CELU: k_gemm_simt<EPI_CELU, ACC><<<grid, THREADS, 0, st>>>(b); break;
    case EPI_CELU_OUT: k_gemm_simt<EPI_CELU_OUT, ACC><<<grid, THREADS, 0, st>>>(b); break;
    case EPI_DCELU: k_gemm_simt<EPI_DCELU, ACC><<<grid, THREADS, 0, st>>>(b); break;
    case EPI_STORE: k_gemm_simt<EPI_STORE, ACC><<<grid, THREADS, 0, st>>>(b); break;
    case EPI_ACCUM: k_gemm_simt<EPI_ACCUM, ACC><<<grid, THREADS, 0, st>>>(b); break;
    }
}

void nnp_launch_gemm_simt(nnp_ctx *c, const GemmBatch &b_in, int epi, int fp64_acc)
{
    GemmBatch b = b_in;
    int tiles = 0, nmax = 0;
    for (int i = 0; i < b.n_groups; ++i) {
        b.tile_off[i] = tiles;
        tiles += nnp_div_up(b.g[i].M, BM);
        if (b.g[i].N > nmax) nmax = b.g[i].N;
    }
    b.tile_off[b.n_groups] = tiles;
    if (tiles == 0) return;
    dim3 grid(tiles, nnp_div_up(nmax, BN));
    if (fp64_acc) launch_simt<double>(c->stream, b, epi, grid);
    else launch_simt<float>(c->stream, b, epi, grid);
    c->launches += 1;
}
