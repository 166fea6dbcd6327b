// lqx harness support: device micro-benchmarks for the roofline denominators --
// FMA-pipe peak (fp32, packed fp32x2, fp64) and a plain vectorised copy.  Not on the hot path.
#include "lqx_internal.cuh"

namespace {

__device__ __forceinline__ void fma2(float2& c, const float2& a, const float2& b) {
    asm("fma.rn.f32x2 %0, %1, %2, %0;"
        : "+l"(reinterpret_cast<unsigned long long&>(c))
        : "l"(reinterpret_cast<const unsigned long long&>(a)), "l"(reinterpret_cast<const unsigned long long&>(b)));
}

// KIND 0: fp32 FMA, 1: fp32x2 packed FMA, 2: fp64 FMA.  16 independent chains per thread.
template <int KIND>
__global__ void __launch_bounds__(256) k_fma_peak(int iters, float seed, double* __restrict__ sink) {
    constexpr int NCH = 16;
    if (KIND == 0) {
        float c[NCH];
        const float a = 1.0f + seed * 1e-7f, b = seed * 1e-9f;
#pragma unroll
        for (int i = 0; i < NCH; ++i) c[i] = (float)(threadIdx.x + i);
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int i = 0; i < NCH; ++i) c[i] = fmaf(c[i], a, b);
        }
        float t = 0.f;
#pragma unroll
        for (int i = 0; i < NCH; ++i) t += c[i];
        if (t == 123.456f) sink[0] = t;
    } else if (KIND == 1) {
        float2 c[NCH];
        const float2 a = make_float2(1.0f + seed * 1e-7f, 1.0f - seed * 1e-7f);
        float2 b = make_float2(seed * 1e-9f, -seed * 1e-9f);
#pragma unroll
        for (int i = 0; i < NCH; ++i) c[i] = make_float2((float)(threadIdx.x + i), (float)i);
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int i = 0; i < NCH; ++i) {
                    // c = c*a + b  written as b' = fma(c, a, b) with roles rotated to keep one chain per i
                    float2 t = b;
                    fma2(t, c[i], a);
                    c[i] = t;
                }
        }
        float t = 0.f;
#pragma unroll
        for (int i = 0; i < NCH; ++i) t += c[i].x + c[i].y;
        if (t == 123.456f) sink[0] = t;
    } else {
        double c[NCH];
        const double a = 1.0 + seed * 1e-12, b = seed * 1e-15;
#pragma unroll
        for (int i = 0; i < NCH; ++i) c[i] = (double)(threadIdx.x + i);
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int i = 0; i < NCH; ++i) c[i] = fma(c[i], a, b);
        }
        double t = 0.0;
#pragma unroll
        for (int i = 0; i < NCH; ++i) t += c[i];
        if (t == 123.456) sink[0] = t;
    }
}

// The same pipes fed the way the lattice kernels feed them: 3x3 complex products on matrices held in registers
// (lqx_internal.cuh mac_nn / mac_na: 108 FMA lane-ops each; fp32 = 54 FFMA2 with broadcast and swapped operands), i.e.
// three DISTINCT register operands per instruction instead of the chain benchmark's one.  What this reaches is the
// FMA rate a product-shaped instruction stream can have at all (register-file ports included).
template <typename T>
__global__ void __launch_bounds__(256) k_product_peak(int iters, T seed, double* __restrict__ sink) {
    Mat3<T> a, b, c;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            a.re[i][j] = (i == j ? T(1) : T(0)) + seed * T(1e-3) * T(threadIdx.x % 7 + i);
            a.im[i][j] = seed * T(1e-3) * T(j + 1);
            b.re[i][j] = (i == j ? T(1) : T(0)) - seed * T(1e-3) * T(i + j);
            b.im[i][j] = seed * T(2e-3) * T(i);
            c.re[i][j] = c.im[i][j] = T(0);
        }
    for (int it = 0; it < iters; ++it) {
        mac_nn(c, a, b);  // c += a b
        mac_na(a, c, b);  // a += c adj(b)
        mac_an(b, a, c);  // b += adj(a) c   (values grow; only the instruction stream matters)
        mac_nn(c, b, a);
    }
    T t = T(0);
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) t += a.re[i][j] + b.im[i][j] + c.re[i][j];
    if (t == T(123.456)) sink[0] = (double)t;
}

__global__ void __launch_bounds__(256) k_copy(size_t n16, const uint4* __restrict__ src, uint4* __restrict__ dst) {
    const size_t step = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += step) dst[i] = src[i];
}

}  // namespace

extern "C" int lqx_bench_fma_peak(lqx_ctx* ctx, int kind, double* lane_ops_per_s) {
    if (!ctx || !lane_ops_per_s || kind < 0 || kind > 4) return LQX_EINVAL;
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const int grid = ctx->num_sms * 8, block = 256, iters = 2048;
    cudaEvent_t e0, e1;
    LQX_CUDA(ctx, cudaEventCreate(&e0));
    LQX_CUDA(ctx, cudaEventCreate(&e1));
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        LQX_CUDA(ctx, cudaEventRecord(e0, ctx->stream));
        if (kind == 0) k_fma_peak<0><<<grid, block, 0, ctx->stream>>>(iters, 1.0f, ctx->d_result + 63);
        else if (kind == 1) k_fma_peak<1><<<grid, block, 0, ctx->stream>>>(iters, 1.0f, ctx->d_result + 63);
        else if (kind == 2) k_fma_peak<2><<<grid, block, 0, ctx->stream>>>(iters, 1.0f, ctx->d_result + 63);
        else if (kind == 3) k_product_peak<float><<<grid, block, 0, ctx->stream>>>(iters, 1e-3f, ctx->d_result + 63);
        else k_product_peak<double><<<grid, block, 0, ctx->stream>>>(iters, 1e-3, ctx->d_result + 63);
        LQX_LAUNCH_CHECK(ctx);
        LQX_CUDA(ctx, cudaEventRecord(e1, ctx->stream));
        LQX_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0.f;
        LQX_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        const double lanes = kind >= 3 ? (double)grid * block * (double)iters * 4.0 * 108.0
                                       : (double)grid * block * (double)iters * 8.0 * 16.0 * (kind == 1 ? 2.0 : 1.0);
        if (rep > 0) best = std::max(best, lanes / (ms * 1e-3));
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *lane_ops_per_s = best;
    return LQX_OK;
}

extern "C" int lqx_bench_copy_peak(lqx_ctx* ctx, size_t bytes, double* bytes_per_s) {
    if (!ctx || !bytes_per_s || bytes < 4096) return LQX_EINVAL;
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t n16 = bytes / 16;
    uint4 *a = nullptr, *b = nullptr;
    if (cudaMalloc(&a, n16 * 16) != cudaSuccess || cudaMalloc(&b, n16 * 16) != cudaSuccess) {
        cudaGetLastError();
        if (a) cudaFree(a);
        return lqx_fail(ctx, LQX_ENOMEM, "copy benchmark buffers");
    }
    cudaMemsetAsync(a, 1, n16 * 16, ctx->stream);
    cudaMemsetAsync(b, 2, n16 * 16, ctx->stream);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    double best = 0.0;
    const int grid = ctx->num_sms * 16;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0, ctx->stream);
        k_copy<<<grid, 256, 0, ctx->stream>>>(n16, a, b);
        ctx->launches++;
        cudaEventRecord(e1, ctx->stream);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0) best = std::max(best, 2.0 * (double)n16 * 16.0 / (ms * 1e-3));
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(a);
    cudaFree(b);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return lqx_cuda_fail(ctx, e, "copy benchmark");
    *bytes_per_s = best;
    return LQX_OK;
}
