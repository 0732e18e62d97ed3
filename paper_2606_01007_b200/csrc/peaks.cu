// tacg_measure_peak: micro-benchmarks of the two units the co-activation kernels saturate, so that
// bench.py divides by MEASURED denominators ("the builder must measure it with a
// tcgen05 kind::i8 micro-benchmark and state the denominator").
//
//   TACG_PEAK_ATOMS_SPREAD  shared-memory atomic increments whose 32 lanes hit 32 different banks
//                           (the best case of a histogram: bank = lane)
//   TACG_PEAK_ATOMS_RANDOM  the same with uniformly random words (the case of a pair histogram)
//   TACG_PEAK_I8_TENSOR     tcgen05.mma kind::i8, M = 128, N = 256, K = 32, issued back to back by one
//                           thread per CTA from shared-memory operands into one TMEM accumulator
//
// Every kernel runs one CTA per SM, is timed with CUDA events after a warm-up launch and also reports its
// own cycle count (clock64), so the result is available per second and per clock and SM.
#include "tacg_common.cuh"
#include "umma.cuh"

namespace {

constexpr int kWords = 32768;   // 128 KB of bins

template <bool RANDOM>
__global__ void __launch_bounds__(1024, 1) atoms_peak_kernel(unsigned* sink, int iters, unsigned long long* cyc) {
    extern __shared__ unsigned bins[];
    const int tid = threadIdx.x, lane = tid & 31;
    for (int i = tid; i < kWords; i += blockDim.x) bins[i] = 0u;
    __syncthreads();
    unsigned a[8];
    unsigned st = tid * 2654435761u + 12345u + blockIdx.x * 97u;
#pragma unroll
    for (int i = 0; i < 8; ++i) { st = st * 1664525u + 1013904223u; a[i] = st >> 7; }
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            a[i] = a[i] * 1664525u + 1013904223u;
            const unsigned r = (a[i] >> 9) & (kWords - 1);
            atomicAdd(&bins[RANDOM ? r : ((r & ~31u) | (unsigned)lane)], 1u);
        }
    }
    __syncthreads();
    const long long t1 = clock64();
    if (tid == 0) cyc[blockIdx.x] = (unsigned long long)(t1 - t0);
    unsigned acc = 0;
    for (int i = tid; i < kWords; i += blockDim.x) acc += bins[i];
    if (acc == 0xdeadbeefu) sink[0] = acc;
}

__global__ void __launch_bounds__(128, 1) i8_peak_kernel(int n_mma, unsigned long long* cyc, unsigned* sink) {
    extern __shared__ __align__(1024) unsigned char ops[];   // A: 128 x 32 bytes, B: 256 x 32 bytes, all ones
    __shared__ uint64_t bar;
    __shared__ uint32_t tbase;
    const int tid = threadIdx.x;
    for (int i = tid; i < (128 * 32 + 256 * 32) / 4; i += blockDim.x) reinterpret_cast<unsigned*>(ops)[i] = 0x01010101u;
    if (tid == 0) { umma::mbar_init(&bar, 1); umma::fence_barrier_init(); }
    __syncthreads();
    if (tid < 32) umma::tmem_alloc(&tbase, 256);
    umma::fence_proxy_async();
    umma::tc_fence_before();
    __syncthreads();
    umma::tc_fence_after();
    const uint32_t tm = tbase;
    if (tid == 0) {
        // MN-major, no swizzle: a core matrix is 8 K-rows x 16 MN bytes; K = 32 is 4 groups of 8 K-rows
        const uint32_t a = umma::smem_u32(ops), b = a + 128 * 32;
        const uint64_t ad = umma::smem_desc_mn_interleave(a, 128 * 8, 128);
        const uint64_t bd = umma::smem_desc_mn_interleave(b, 256 * 8, 128);
        const uint32_t idesc = umma::idesc_u8_mn(128, 256);
        const long long t0 = clock64();
        for (int i = 0; i < n_mma; ++i) umma::mma_i8_ss(tm, ad, bd, idesc, i > 0);
        umma::mma_commit(&bar);
        umma::mbar_wait(&bar, 0);
        cyc[blockIdx.x] = (unsigned long long)(clock64() - t0);
    }
    __syncthreads();
    umma::tc_fence_after();
    if (tid < 32) {
        uint32_t v[16];
        umma::tmem_ld_32x32b_x16(tm, v);
        umma::tmem_ld_wait();
        if (blockIdx.x == 0 && tid == 0) sink[0] = v[0];    // = 32 * n_mma: every product is 1 x 1
    }
    __syncthreads();
    if (tid < 32) umma::tmem_dealloc(tm, 256);
}

}  // namespace

extern "C" int tacg_measure_peak(tacg_ctx* ctx, int which, double* per_second, double* per_clk_sm) {
    if (!ctx || !per_second || !per_clk_sm) return TACG_ERR_NULL;
    if (which < 0 || which > TACG_PEAK_I8_TENSOR) return TACG_ERR_SHAPE;
    TACG_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    const int sms = ctx->sm_count;
    unsigned long long* cyc = nullptr;
    unsigned* sink = nullptr;
    TACG_CUDA_TRY(ctx, cudaMalloc(&cyc, sizeof(unsigned long long) * sms));
    TACG_CUDA_TRY(ctx, cudaMalloc(&sink, 2 * sizeof(unsigned)));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    double units = 0.0;      // increments (or multiply-adds x 2) of one SM in the timed launch
    int rc = TACG_OK;
    auto launch = [&](bool timed) -> cudaError_t {
        if (timed) cudaEventRecord(e0, ctx->stream);
        if (which == TACG_PEAK_I8_TENSOR) {
            const int n = timed ? 20000 : 100;
            const int smem = 128 * 32 + 256 * 32 + 1024;
            cudaFuncSetAttribute(i8_peak_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
            i8_peak_kernel<<<sms, 128, smem, ctx->stream>>>(n, cyc, sink);
            units = 2.0 * 128 * 256 * 32 * n;
        } else {
            const int iters = timed ? 2000 : 10;
            if (which == TACG_PEAK_ATOMS_RANDOM) {
                cudaFuncSetAttribute(atoms_peak_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kWords * 4);
                atoms_peak_kernel<true><<<sms, 1024, kWords * 4, ctx->stream>>>(sink, iters, cyc);
            } else {
                cudaFuncSetAttribute(atoms_peak_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kWords * 4);
                atoms_peak_kernel<false><<<sms, 1024, kWords * 4, ctx->stream>>>(sink, iters, cyc);
            }
            units = 1024.0 * 8 * iters;
        }
        if (timed) cudaEventRecord(e1, ctx->stream);
        return cudaGetLastError();
    };
    cudaError_t err = launch(false);
    if (err == cudaSuccess) err = launch(true);
    if (err == cudaSuccess) err = cudaStreamSynchronize(ctx->stream);
    if (err != cudaSuccess) {
        snprintf(ctx->detail, sizeof(ctx->detail), "tacg_measure_peak: %s", cudaGetErrorString(err));
        rc = TACG_ERR_CUDA;
    } else {
        ctx->launches += 2;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        std::vector<unsigned long long> h(sms);
        cudaMemcpy(h.data(), cyc, sizeof(unsigned long long) * sms, cudaMemcpyDeviceToHost);
        unsigned long long mx = 1;
        for (int i = 0; i < sms; ++i) mx = h[i] > mx ? h[i] : mx;
        *per_second = units * sms / (ms * 1e-3);
        *per_clk_sm = units / (double)mx;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(cyc);
    cudaFree(sink);
    return rc;
}
