// lqx_norm2_noalloc: norm2 of a field (Listing 1, the norm2() of the Jacobi routine)
// for callers that cannot allocate device memory -- code under CUDA graph capture, serving loops, harnesses that forbid
// cudaMalloc.  The existing lqx_norm2 takes its reduction scratch (per-CTA partial sums and the last-block ticket) from
// the context, which grows it with cudaMalloc on demand (lqx_ensure_partials); this entry point takes it from a
// file-scope __device__ array of fixed size instead, and calls no cudaMalloc / cudaFree / allocating library routine.
//
//  * The array is LQX_NOALLOC_SCRATCH_BYTES (64 KB + 256 B) of global memory on EVERY GPU that loads the library,
//    held until the process exits.
//  * One partial per CTA and kSitesPerCta sites per CTA fix the largest lattice: LQX_NOALLOC_MAX_SITES = 2^24 sites
//    (48^3 x 96 = 10.6 M fits).  A larger lattice is rejected with LQX_EINVAL and a message; nothing is launched.
//  * In host code the array's NAME is a host-side stand-in, not a device address.  The address a kernel may be given
//    comes from cudaGetSymbolAddress, asked once per device with that device current (scratch_for below).
//  * All calls share the array, and it keeps the last call's contents.  The partials need no clearing (a call writes
//    slots [0, grid) before its last CTA reads exactly those); the ticket must start at zero and is cleared on the
//    stream in front of every launch.  Two calls that overlap on the GPU (different streams or contexts on one
//    device) race on it: serialise them.
//  * The summation tree is a function of the lattice volume only (not of the SM count), so the result is the same
//    from run to run and from GPU to GPU; it differs from lqx_norm2's tree, i.e. the two agree to rounding.
#include <mutex>

#include "lqx_internal.cuh"

namespace {

constexpr int kThreads = 256;
constexpr int kSitesPerThread = 8;
constexpr int kSitesPerCta = kThreads * kSitesPerThread;  // 2048
constexpr int kMaxCtas = 8192;                            // one fp64 partial each: 64 KB
constexpr size_t kTicketOffset = (size_t)kMaxCtas * sizeof(double);
static_assert((long long)kMaxCtas * kSitesPerCta == LQX_NOALLOC_MAX_SITES, "include/lqx.h states the maximum");
static_assert(kTicketOffset + 256 == LQX_NOALLOC_SCRATCH_BYTES, "include/lqx.h states the size");

// [0, 64 KB): per-CTA partial sums; [64 KB, +4): the last-block ticket
static __device__ __align__(256) unsigned char g_noalloc_scratch[LQX_NOALLOC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
unsigned char* g_scratch_addr[kMaxDevices];  // device address of g_noalloc_scratch on each device, nullptr = not asked yet

// device address of the scratch array on ctx's device (which the caller has made current)
int scratch_for(lqx_ctx* ctx, unsigned char** addr) {
    if (ctx->device < 0 || ctx->device >= kMaxDevices) return lqx_fail(ctx, LQX_EINVAL, "lqx_norm2_noalloc: device ordinal beyond the set-up table");
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_addr[ctx->device]) {
        void* p = nullptr;
        LQX_CUDA(ctx, cudaGetSymbolAddress(&p, g_noalloc_scratch));
        if (!p) return lqx_fail(ctx, LQX_ECUDA, "cudaGetSymbolAddress(g_noalloc_scratch) returned no address");
        g_scratch_addr[ctx->device] = static_cast<unsigned char*>(p);
    }
    *addr = g_scratch_addr[ctx->device];
    return LQX_OK;
}

// CTA b sums the sites [b * 2048, (b + 1) * 2048): thread t takes b * 2048 + k * 256 + t, k = 0..7 (coalesced),
// |z|^2 accumulated in fp64 in two chains per site as k_norm2 does; then the deterministic CTA tree, one partial per
// CTA, and the CTA that draws the last ticket adds the partials in a fixed order and writes out[0].
template <typename T, int NREAL>
__global__ void __launch_bounds__(kThreads) k_norm2_noalloc(int V, const T* __restrict__ f, double* __restrict__ partials,
                                                            unsigned int* __restrict__ ticket, double* __restrict__ out) {
    double acc[1] = {0.0};
    const int base = blockIdx.x * kSitesPerCta + threadIdx.x;
#pragma unroll 2
    for (int k = 0; k < kSitesPerThread; ++k) {
        const int s = base + k * kThreads;
        if (s < V) {
            T r[NREAL];
            load_site<T, NREAL>(f, s, r);
            double t0 = 0.0, t1 = 0.0;
#pragma unroll
            for (int j = 0; j < NREAL; j += 2) {
                t0 = fma((double)r[j], (double)r[j], t0);
                t1 = fma((double)r[j + 1], (double)r[j + 1], t1);
            }
            acc[0] += t0 + t1;
        }
    }
    block_reduce_finish<1>(acc, partials, ticket, out);
}

template <typename T>
int launch(lqx_ctx* ctx, const lqx_field* f, int grid, double* partials, unsigned int* ticket, double* out) {
    const int V = ctx->geo.V;
    const T* p = (const T*)f->data;
    switch ((int)f->kind) {
        case LQX_COMPLEX: k_norm2_noalloc<T, 2><<<grid, kThreads, 0, ctx->stream>>>(V, p, partials, ticket, out); break;
        case LQX_COLORVEC: k_norm2_noalloc<T, 6><<<grid, kThreads, 0, ctx->stream>>>(V, p, partials, ticket, out); break;
        case LQX_COLORMAT: k_norm2_noalloc<T, 18><<<grid, kThreads, 0, ctx->stream>>>(V, p, partials, ticket, out); break;
        case LQX_FERMION: k_norm2_noalloc<T, 24><<<grid, kThreads, 0, ctx->stream>>>(V, p, partials, ticket, out); break;
        default: return lqx_fail(ctx, LQX_ETYPE, "lqx_norm2_noalloc: unknown field kind");
    }
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}

}  // namespace

extern "C" int lqx_norm2_noalloc(const lqx_field* f, double* out_dev) {
    if (!f || !out_dev) return LQX_EINVAL;
    lqx_ctx* ctx = f->ctx;
    const long long V = ctx->geo.V;
    if (V > LQX_NOALLOC_MAX_SITES)
        return lqx_fail(ctx, LQX_EINVAL, "lqx_norm2_noalloc: the lattice has more sites than the static scratch serves (LQX_NOALLOC_MAX_SITES = 16777216)");
    if ((uintptr_t)out_dev % sizeof(double)) return lqx_fail(ctx, LQX_EINVAL, "lqx_norm2_noalloc: out_dev must be 8-byte aligned");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    unsigned char* scratch = nullptr;
    const int rc = scratch_for(ctx, &scratch);
    if (rc) return rc;
    double* partials = reinterpret_cast<double*>(scratch);
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + kTicketOffset);
    const int grid = (int)((V + kSitesPerCta - 1) / kSitesPerCta);  // >= 1, <= kMaxCtas
    // the ticket counts the CTAs that have stored their partial: it must be zero when the grid starts, whatever an
    // earlier (possibly failed) call left there
    LQX_CUDA(ctx, cudaMemsetAsync(ticket, 0, sizeof(unsigned int), ctx->stream));
    return f->prec == LQX_F32 ? launch<float>(ctx, f, grid, partials, ticket, out_dev) : launch<double>(ctx, f, grid, partials, ticket, out_dev);
}
