// Roofline denominators measured on the device the library runs on ("TF32 tcgen05 peak must be
// measured by the builder ... fp32 FMA peak and SFU peak - both to be microbenchmarked and committed next to the ncu
// reports").  Three micro-kernels, no memory traffic inside the timed loops:
//   * fp32 FMA:   8 independent FFMA chains per thread, every SM full           -> TFLOP/s (2 flops per FMA)
//   * MUFU ex2:   8 independent ex2.approx chains per thread                     -> G ops/s
//   * tcgen05:    one CTA per SM issues back-to-back tcgen05.mma.kind::tf32 M128 N256 K8 on resident shared-memory /
//                 tensor-memory operands (both operand forms: A from shared memory, and A from TMEM as the MLP GEMMs
//                 of mlp_tc.cu use it)                                            -> dense TF32 TFLOP/s
// nnp_measure_peaks is a diagnostic entry of the C-ABI (include/nnp.h); nothing on the hot path calls it.
#include <cuda_runtime.h>
#include <stdint.h>

#include "nnp_internal.cuh"

namespace {

constexpr int kChains = 8;

__global__ void __launch_bounds__(256) k_peak_fma(int iters, float a, float b, float *out)
{
    float x[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) x[c] = (float)(threadIdx.x + c) * 1e-3f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) x[c] = fmaf(x[c], a, b);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < kChains; ++c) s += x[c];
    if (s == 123.456f) out[0] = s; // never true: keeps the chains alive
}

__global__ void __launch_bounds__(256) k_peak_mufu(int iters, float *out)
{
    float x[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) x[c] = (float)(threadIdx.x + c) * 1e-3f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(x[c]) : "f"(-x[c])); // 2^-x stays in (0.5, 1]
        }
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < kChains; ++c) s += x[c];
    if (s == 123.456f) out[0] = s;
}

// ---- tcgen05 (same operand layout as mlp_tc.cu: K-major tiles of 128-byte rows, 128-byte swizzle)
constexpr int PK_M = 128, PK_N = 256, PK_K = 8;
constexpr int PK_A_BYTES = PK_M * 128, PK_B_BYTES = PK_N * 128;
constexpr int PK_SMEM = 1024 + PK_A_BYTES + PK_B_BYTES + 64;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint64_t kmajor_sw128_desc(uint32_t smem_addr)
{
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr >> 4) & 0x3fff);
    d |= (uint64_t)1 << 16;
    d |= (uint64_t)(1024 >> 4) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}

// TS = false: D[tmem] += A[smem] . B[smem]^T;  TS = true: A from tensor memory (columns 256..287)
template <bool TS>
__global__ void __launch_bounds__(128, 1) k_peak_tf32(int n_groups, int mma_n, long long *cycles)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t a_smem = base, b_smem = base + PK_A_BYTES, bar = b_smem + PK_B_BYTES, slot = bar + 8;
    const int warp = threadIdx.x >> 5;
    for (uint32_t off = threadIdx.x * 16; off < (uint32_t)(PK_A_BYTES + PK_B_BYTES); off += 128 * 16)
        asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(base + off), "r"(0u) : "memory");
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(slot) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); // the zero-filled operands are read by the tensor core
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    uint32_t tmem;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem) : "r"(slot));
    if (TS) { // zero the A operand in tensor memory: this warp's 32 lanes x 32 columns
        const uint32_t taddr = tmem + ((uint32_t)(warp * 32) << 16) + 256u;
#pragma unroll
        for (int c = 0; c < 32; c += 8)
            asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %1, %1, %1, %1, %1, %1, %1};" ::"r"(taddr + c), "r"(0u) : "memory");
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    }
    if (threadIdx.x == 0) {
        const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(mma_n >> 3) << 17) | ((uint32_t)(PK_M >> 4) << 24);
        const uint64_t da = kmajor_sw128_desc(a_smem), db = kmajor_sw128_desc(b_smem);
        const long long t0 = clock64();
        for (int g = 0; g < n_groups; ++g) {
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint64_t koff = (uint64_t)(k * PK_K * 4 >> 4);
                const uint32_t acc_on = (g | k) ? 1u : 0u;
                if (TS)
                    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}" ::"r"(tmem),
                                 "r"(tmem + 256u + k * PK_K), "l"(db + koff), "r"(idesc), "r"(acc_on)
                                 : "memory");
                else
                    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem),
                                 "l"(da + koff), "l"(db + koff), "r"(idesc), "r"(acc_on)
                                 : "memory");
            }
        }
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
        uint32_t done = 0;
        for (uint32_t spin = 0; spin < (1u << 28) && !done; ++spin)
            asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                         : "=r"(done)
                         : "r"(bar)
                         : "memory");
        cycles[blockIdx.x] = done ? clock64() - t0 : -1;
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
    }
}

template <class F>
float best_ms(F launch, int reps)
{
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float best = 1e30f;
    for (int r = 0; r < reps; ++r) {
        cudaEventRecord(e0);
        launch();
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best) best = ms; // the first launch is the warm-up
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return best;
}

} // namespace

extern "C" int nnp_measure_peaks(int device, double *h_out /* [NNP_N_PEAKS] */)
{
    if (!h_out) return NNP_EINVAL;
    if (cudaSetDevice(device) != cudaSuccess) return NNP_ECUDA;
    int sms = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (sms <= 0) return NNP_ECUDA;
    float *d_out = nullptr;
    long long *d_cyc = nullptr;
    if (cudaMalloc(&d_out, 16) != cudaSuccess || cudaMalloc(&d_cyc, sizeof(long long) * sms) != cudaSuccess) return NNP_ENOMEM;
    const int blocks = sms * 8, threads = 256, iters = 4096;
    const double alu_ops = (double)blocks * threads * (double)iters * 8.0 * kChains;
    const float ms_fma = best_ms([&] { k_peak_fma<<<blocks, threads>>>(iters, 0.999f, 1e-3f, d_out); }, 6);
    const float ms_mufu = best_ms([&] { k_peak_mufu<<<blocks, threads>>>(iters / 4, d_out); }, 6);
    h_out[0] = 2.0 * alu_ops / (ms_fma * 1e-3) * 1e-12; // TFLOP/s
    h_out[1] = alu_ops / 4.0 / (ms_mufu * 1e-3) * 1e-9; // G ops/s
    const int n_groups = 8192; // x 4 MMAs of M128 N256 K8
    const double mma_flops = 2.0 * PK_M * PK_N * PK_K * 4.0 * n_groups * sms;
    cudaFuncSetAttribute(k_peak_tf32<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, PK_SMEM);
    cudaFuncSetAttribute(k_peak_tf32<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, PK_SMEM);
    long long cyc[2] = {0, 0};
    const float ms_ss = best_ms([&] { k_peak_tf32<false><<<sms, 128, PK_SMEM>>>(n_groups, PK_N, d_cyc); }, 4);
    cudaMemcpy(&cyc[0], d_cyc, sizeof(long long), cudaMemcpyDeviceToHost);
    const float ms_ts = best_ms([&] { k_peak_tf32<true><<<sms, 128, PK_SMEM>>>(n_groups, PK_N, d_cyc); }, 4);
    cudaMemcpy(&cyc[1], d_cyc, sizeof(long long), cudaMemcpyDeviceToHost);
    h_out[2] = mma_flops / (ms_ss * 1e-3) * 1e-12;
    h_out[3] = mma_flops / (ms_ts * 1e-3) * 1e-12;
    h_out[4] = cyc[0] > 0 ? (double)cyc[0] / (4.0 * n_groups) : -1.0; // SM cycles per MMA instruction (M128 N256 K8)
    h_out[5] = cyc[1] > 0 ? (double)cyc[1] / (4.0 * n_groups) : -1.0;
    // cycles per MMA instruction (A in tensor memory) against the N extent: NNP_PEAK_N_LIST columns 64, 96, ..., 256
    for (int q = 0; q < 7; ++q) {
        const int mma_n = 64 + 32 * q;
        k_peak_tf32<true><<<sms, 128, PK_SMEM>>>(n_groups / 4, mma_n, d_cyc);
        long long c = 0;
        cudaMemcpy(&c, d_cyc, sizeof(long long), cudaMemcpyDeviceToHost);
        h_out[6 + q] = c > 0 ? (double)c / (double)n_groups : -1.0;
    }
    cudaFree(d_out);
    cudaFree(d_cyc);
    return cudaGetLastError() == cudaSuccess ? NNP_OK : NNP_ECUDA;
}
