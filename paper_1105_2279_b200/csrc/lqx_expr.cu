// lqx expression catalogue and standalone global reductions (a9).
// Every entry point is one pass over HBM: the whole expression, shift included, is evaluated per
// site with no temporaries (the paper's evaluate()).  One thread owns one
// site; its operands arrive as 128-bit loads from the blocked SoA store (lqx_internal.cuh), so a
// warp moves 512 contiguous bytes per instruction.
#include "lqx_internal.cuh"

namespace {

__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }

int check_same(lqx_ctx** ctx_out, std::initializer_list<const lqx_field*> fs) {
    lqx_ctx* ctx = nullptr;
    lqx_prec prec = LQX_F32;
    for (const lqx_field* f : fs) {
        if (!f) return LQX_EINVAL;
        if (!ctx) {
            ctx = f->ctx;
            prec = f->prec;
        } else {
            if (f->ctx != ctx) return lqx_fail(ctx, LQX_EGEOM, "operands belong to different contexts");
            if (f->prec != prec) return lqx_fail(ctx, LQX_ETYPE, "mixed precision operands");
        }
    }
    *ctx_out = ctx;
    return LQX_OK;
}

// ---------------------------------------------------------------------------------------------
// flat elementwise kernels over the raw storage (layout-agnostic; pad lanes included, they are
// never read for results).  mode 0: r = a ; 1: r = a + k*b ; 2: r = k*a ; 3: r = a / k
// ---------------------------------------------------------------------------------------------
template <typename T, int MODE, bool INPLACE>
__global__ void __launch_bounds__(256) k_flat(size_t nvec, T k, typename KPtr<T, INPLACE>::in a, typename KPtr<T, INPLACE>::in b,
                                              typename KPtr<T, INPLACE>::out r) {
    typedef typename Vec128<T>::type V;
    constexpr int W = Vec128<T>::W;
    const size_t step = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += step) {
        T va[W], vb[W], vr[W];
        unpack(reinterpret_cast<const V*>(a)[i], va);
        if (MODE == 1) unpack(reinterpret_cast<const V*>(b)[i], vb);
#pragma unroll
        for (int j = 0; j < W; ++j) {
            if (MODE == 0) vr[j] = va[j];
            if (MODE == 1) vr[j] = fma(k, vb[j], va[j]);
            if (MODE == 2) vr[j] = k * va[j];
            if (MODE == 3) vr[j] = va[j] / k;
        }
        reinterpret_cast<V*>(r)[i] = pack(vr);
    }
}

template <typename T, int MODE>
int flat_launch(lqx_ctx* ctx, lqx_field* r, const lqx_field* a, const lqx_field* b, double k) {
    const size_t n = (size_t)ctx->geo.Vpad * 2 * (int)r->kind;
    const size_t nvec = n / Vec128<T>::W;
    const int block = 256;
    size_t want = (nvec + block - 1) / block;
    int grid = (int)std::min<size_t>(want, (size_t)ctx->num_sms * 16);
    if (grid < 1) grid = 1;
    // in place (r is a or b, reading A21): the instantiation without __restrict__ / read-only loads
    const bool inplace = lqx_identical(r, a) || (b && lqx_identical(r, b));
    LqxTimed timed(ctx, LQX_K_CATALOGUE);
    if (inplace) k_flat<T, MODE, true><<<grid, block, 0, ctx->stream>>>(nvec, (T)k, (const T*)a->data, b ? (const T*)b->data : nullptr, (T*)r->data);
    else k_flat<T, MODE, false><<<grid, block, 0, ctx->stream>>>(nvec, (T)k, (const T*)a->data, b ? (const T*)b->data : nullptr, (T*)r->data);
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}

template <int MODE>
int flat_dispatch(lqx_field* r, const lqx_field* a, const lqx_field* b, double k) {
    lqx_ctx* ctx;
    int rc = b ? check_same(&ctx, {r, a, b}) : check_same(&ctx, {r, a});
    if (rc) return rc;
    if (r->kind != a->kind || (b && b->kind != a->kind)) return lqx_fail(ctx, LQX_ETYPE, "field kinds differ");
    if ((lqx_same(r, a) && !lqx_identical(r, a)) || (b && lqx_same(r, b) && !lqx_identical(r, b)))
        return lqx_fail(ctx, LQX_EALIAS, "destination partially overlaps an operand");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    return r->prec == LQX_F32 ? flat_launch<float, MODE>(ctx, r, a, b, k) : flat_launch<double, MODE>(ctx, r, a, b, k);
}

// ---------------------------------------------------------------------------------------------
// shift and form (iii): one thread per site; the shifted operand is the whole site object at the
// periodic neighbour ("shift ... reads its operand through a site table" -- here the
// index is computed).  AX = false: r = shift(b);  AX = true: r = alpha*a - shift(b)
// ---------------------------------------------------------------------------------------------
template <typename T, int NREAL, bool AX, bool INPLACE>
__global__ void __launch_bounds__(128) k_shift(const __grid_constant__ Geo g, int dir, int mu, T alpha, typename KPtr<T, INPLACE>::in a,
                                               const T* __restrict__ b, typename KPtr<T, INPLACE>::out r) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.V) return;
    int x[4];
    site_coords(g, s, x);
    const int n = dir > 0 ? nbr_fwd(g, s, x, mu) : nbr_bwd(g, s, x, mu);
    T vb[NREAL];
    load_site<T, NREAL>(b, n, vb);
    if (AX) {
        T va[NREAL];
        load_site<T, NREAL, INPLACE>(a, s, va);
#pragma unroll
        for (int j = 0; j < NREAL; ++j) vb[j] = mul_rn(alpha, va[j]) - vb[j];  // alpha*A rounded once, as written
    }
    store_site<T, NREAL>(r, s, vb);
}

template <typename T, bool AX>
int shift_launch(lqx_ctx* ctx, lqx_field* r, double alpha, const lqx_field* a, const lqx_field* b, int dir, int mu) {
    const Geo& g = ctx->geo;
    const int block = 128, grid = (g.V + block - 1) / block;
    const T* pa = a ? (const T*)a->data : nullptr;
    const T* pb = (const T*)b->data;
    T* pr = (T*)r->data;
    const bool inplace = AX && a && lqx_identical(r, a);  // form iii may overwrite its UNshifted operand (A21)
    LqxTimed timed(ctx, LQX_K_CATALOGUE);
#define LQX_SHIFT_LAUNCH(NREAL)                                                                                   \
    if (inplace) k_shift<T, NREAL, AX, AX><<<grid, block, 0, ctx->stream>>>(g, dir, mu, (T)alpha, pa, pb, pr);     \
    else k_shift<T, NREAL, AX, false><<<grid, block, 0, ctx->stream>>>(g, dir, mu, (T)alpha, pa, pb, pr);
    switch ((int)r->kind) {
        case LQX_COMPLEX: LQX_SHIFT_LAUNCH(2) break;
        case LQX_COLORVEC: LQX_SHIFT_LAUNCH(6) break;
        case LQX_COLORMAT: LQX_SHIFT_LAUNCH(18) break;
        default: LQX_SHIFT_LAUNCH(24) break;
    }
#undef LQX_SHIFT_LAUNCH
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}

// ---------------------------------------------------------------------------------------------
// site-local matrix forms: one thread per site, all operands of the site in registers
// ---------------------------------------------------------------------------------------------
// form (i) R = A*B + C*adj(D)
template <typename T, bool INPLACE>
__global__ void __launch_bounds__(128) k_mm_plus_madj(int V, typename KPtr<T, INPLACE>::in a, typename KPtr<T, INPLACE>::in b,
                                                      typename KPtr<T, INPLACE>::in c, typename KPtr<T, INPLACE>::in d,
                                                      typename KPtr<T, INPLACE>::out r) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= V) return;
    const Mat3<T> ma = load_mat<T, INPLACE>(a, s), mb = load_mat<T, INPLACE>(b, s);
    const Mat3<T> mc = load_mat<T, INPLACE>(c, s), md = load_mat<T, INPLACE>(d, s);
    Mat3<T> acc = mul_nn(ma, mb);
    mac_na(acc, mc, md);
    store_mat(r, s, acc);
}
// form (ii) c = trace(A*B) = sum_ik A_ik B_ki
template <typename T>
__global__ void __launch_bounds__(128) k_trace_mm(int V, const T* __restrict__ a, const T* __restrict__ b, T* __restrict__ c) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= V) return;
    const Mat3<T> ma = load_mat(a, s), mb = load_mat(b, s);
    T re = T(0), im = T(0);
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            re = fma(ma.re[i][k], mb.re[k][i], re);
            re = fma(-ma.im[i][k], mb.im[k][i], re);
            im = fma(ma.re[i][k], mb.im[k][i], im);
            im = fma(ma.im[i][k], mb.re[k][i], im);
        }
    const T out[2] = {re, im};
    store_site<T, 2>(c, s, out);
}
// form (iv) w = M*v per spin component
template <typename T, int NSPIN, bool INPLACE>
__global__ void __launch_bounds__(128) k_mat_vec(int V, const T* __restrict__ m, typename KPtr<T, INPLACE>::in v,
                                                 typename KPtr<T, INPLACE>::out w) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= V) return;
    const Mat3<T> mm = load_mat(m, s);
    Vec3<T> vv[NSPIN], ww[NSPIN];
    load_vecs<T, NSPIN, INPLACE>(v, s, vv);
#pragma unroll
    for (int a = 0; a < NSPIN; ++a) {
#pragma unroll
        for (int i = 0; i < 3; ++i) ww[a].re[i] = ww[a].im[i] = T(0);
        mac_mv(ww[a], mm, vv[a]);
    }
    store_vecs<T, NSPIN>(w, s, ww);
}

// ---------------------------------------------------------------------------------------------
// standalone reductions: one launch.  Each thread accumulates in fp64 over a grid-stride loop of
// sites with a FIXED grid, then the deterministic block tree + last-block finish
// (lqx_internal.cuh) writes the result straight into pinned host memory.
// ---------------------------------------------------------------------------------------------
template <typename T, int NREAL>
__global__ void __launch_bounds__(256, 8) k_norm2(int V, const T* __restrict__ f, double* __restrict__ partials, unsigned int* ticket,
                                               double* __restrict__ out) {
    double acc[1] = {0.0};
    const int step = gridDim.x * blockDim.x;
    for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < V; s += step) {
        T r[NREAL];
        load_site<T, NREAL>(f, s, r);
        double t0 = 0.0, t1 = 0.0;  // two chains per site object
#pragma unroll
        for (int j = 0; j < NREAL; j += 2) {
            t0 = fma((double)r[j], (double)r[j], t0);
            t1 = fma((double)r[j + 1], (double)r[j + 1], t1);
        }
        acc[0] += t0 + t1;
    }
    block_reduce_finish<1>(acc, partials, ticket, out);
}
// sum over sites of the site object -> NREAL doubles in QDP order.
// A warp OWNS one 128-bit chunk position q of the site object (the blocked layout keeps chunk q of 32 consecutive
// sites contiguous) and walks over the 32-site blocks: a thread then accumulates only the W = 4 (fp32) or 2 (fp64)
// reals of its chunk -- 4 fp64 accumulators instead of the 2*kind of a thread-per-site loop (36 registers for a
// colour matrix, which halved the occupancy: 38 us against 31 us for norm2 on the same 151 MB) -- and has UNR
// independent 128-bit loads in flight.  SUB warps share a chunk position inside a CTA and are combined through
// shared memory in a fixed order, so one CTA still produces one partial per component.  The pad lanes of the last
// block are zero by the layout's invariant, so whole blocks are summed.
template <typename T, int NREAL, int SUB>
__global__ void __launch_bounds__(32 * SUB * ((NREAL + Vec128<T>::W - 1) / Vec128<T>::W), 64 / (SUB * ((NREAL + Vec128<T>::W - 1) / Vec128<T>::W)))
    k_sum(int nblk, const T* __restrict__ f, double* __restrict__ partials, unsigned int* ticket, double* __restrict__ out) {
    typedef typename Vec128<T>::type V128;
    constexpr int W = Vec128<T>::W, NFULL = NREAL / W, NQ = (NREAL + W - 1) / W, UNR = 4;
    __shared__ double sh[SUB][NQ * W];
    __shared__ bool last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int q = warp % NQ, sub = warp / NQ;
    const int nblocks = gridDim.x;
    double acc[W];
#pragma unroll
    for (int r = 0; r < W; ++r) acc[r] = 0.0;
    const int stride = nblocks * SUB;
    int b = blockIdx.x * SUB + sub;
    if (q < NFULL) {  // a full chunk: 128 bits per site
        static_assert((32 * NREAL * sizeof(T)) % sizeof(V128) == 0, "block pitch");
        constexpr size_t BLK = (size_t)32 * NREAL * sizeof(T) / sizeof(V128);  // block pitch in 128-bit units
        const V128* p = reinterpret_cast<const V128*>(f + (size_t)q * 32 * W) + lane;
        for (; b + (UNR - 1) * stride < nblk; b += UNR * stride) {
            V128 v[UNR];
#pragma unroll
            for (int k = 0; k < UNR; ++k) v[k] = __ldg(p + (size_t)(b + k * stride) * BLK);
#pragma unroll
            for (int k = 0; k < UNR; ++k) {
                T r[W];
                unpack(v[k], r);
#pragma unroll
                for (int j = 0; j < W; ++j) acc[j] += (double)r[j];
            }
        }
        for (; b < nblk; b += stride) {
            T r[W];
            unpack(__ldg(p + (size_t)b * BLK), r);
#pragma unroll
            for (int j = 0; j < W; ++j) acc[j] += (double)r[j];
        }
    } else {  // fp32 only: the trailing (re, im) pair, 64 bits per site
        constexpr size_t BLK = (size_t)32 * NREAL * sizeof(T) / sizeof(float2);
        const float2* p = reinterpret_cast<const float2*>(f + (size_t)NFULL * 32 * W) + lane;
        for (; b + (UNR - 1) * stride < nblk; b += UNR * stride) {
            float2 v[UNR];
#pragma unroll
            for (int k = 0; k < UNR; ++k) v[k] = __ldg(p + (size_t)(b + k * stride) * BLK);
#pragma unroll
            for (int k = 0; k < UNR; ++k) {
                acc[0] += (double)v[k].x;
                acc[1] += (double)v[k].y;
            }
        }
        for (; b < nblk; b += stride) {
            const float2 v = __ldg(p + (size_t)b * BLK);
            acc[0] += (double)v.x;
            acc[1] += (double)v.y;
        }
    }
#pragma unroll
    for (int r = 0; r < W; ++r) {
        double t = acc[r];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (lane == 0) sh[sub][q * W + r] = t;
    }
    __syncthreads();
    static_assert(NREAL <= 32, "one warp stores the CTA's partials");
    if (warp == 0) {
        if (lane < NREAL) {
            double t = sh[0][lane];
#pragma unroll
            for (int k = 1; k < SUB; ++k) t += sh[k][lane];
            partials[(size_t)lane * nblocks + blockIdx.x] = t;
        }
        __syncwarp();
        if (lane == 0) {  // release-only ticket, as in block_reduce_finish
            unsigned int t;
            asm volatile("atom.release.gpu.global.add.u32 %0, [%1], 1;" : "=r"(t) : "l"(ticket) : "memory");
            last = (t == (unsigned)(nblocks - 1));
        }
    }
    __syncthreads();
    if (!last) return;
    __threadfence();  // acquire side, paid by the one finishing CTA
    for (int c = warp; c < NREAL; c += (int)(blockDim.x >> 5)) {  // one warp per component, fixed order
        const double* pc = partials + (size_t)c * nblocks;
        double t0 = 0.0, t1 = 0.0, t2 = 0.0, t3 = 0.0;
        int i = lane;
        for (; i + 96 < nblocks; i += 128) {
            const double a0 = __ldcg(pc + i), a1 = __ldcg(pc + i + 32), a2 = __ldcg(pc + i + 64), a3 = __ldcg(pc + i + 96);
            t0 += a0, t1 += a1, t2 += a2, t3 += a3;
        }
        for (; i < nblocks; i += 32) t0 += __ldcg(pc + i);
        double t = (t0 + t1) + (t2 + t3);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (lane == 0) out[c] = t;
    }
    __syncthreads();
    if (threadIdx.x == 0) *ticket = 0u;  // ready for the next launch on this stream
}
// sum_x tr M(x): diagonal elements (0,0),(1,1),(2,2) = QDP reals 0,1 / 8,9 / 16,17
template <typename T>
__global__ void __launch_bounds__(256) k_trace(int V, const T* __restrict__ m, double* __restrict__ partials, unsigned int* ticket,
                                               double* __restrict__ out) {
    typedef typename Vec128<T>::type V128;
    constexpr int W = Vec128<T>::W;
    double acc[2] = {0.0, 0.0};
    const int step = gridDim.x * blockDim.x;
    for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < V; s += step) {
        // only the chunks that hold diagonal elements are touched: fp32 chunks 0, 2, 4; fp64 chunks 0, 4, 8
        const T* blk = m + (size_t)(s >> 5) * (32 * 18);
        const int lane = s & 31;
        if (W == 4) {
            T c0[W], c2[W];
            unpack(__ldg(reinterpret_cast<const V128*>(blk) + lane), c0);
            unpack(__ldg(reinterpret_cast<const V128*>(blk) + 2 * 32 + lane), c2);
            const float2 c4 = __ldg(reinterpret_cast<const float2*>(blk + 4 * 32 * 4) + lane);
            acc[0] += (double)c0[0] + (double)c2[0] + (double)c4.x;
            acc[1] += (double)c0[1] + (double)c2[1] + (double)c4.y;
        } else {
            T d0[W], d1[W], d2[W];
            unpack(__ldg(reinterpret_cast<const V128*>(blk) + lane), d0);
            unpack(__ldg(reinterpret_cast<const V128*>(blk) + 4 * 32 + lane), d1);
            unpack(__ldg(reinterpret_cast<const V128*>(blk) + 8 * 32 + lane), d2);
            acc[0] += (double)d0[0] + (double)d1[0] + (double)d2[0];
            acc[1] += (double)d0[1] + (double)d1[1] + (double)d2[1];
        }
    }
    block_reduce_finish<2>(acc, partials, ticket, out);
}

int reduce_grid(const lqx_ctx* ctx, int sites_per_thread, int ctas_per_sm = 8) {
    // fixed function of V (and the SM count) only => deterministic summation tree; the cap is the number of CTAs
    // that are resident at once, so that the grid is one wave
    long want = ((long)ctx->geo.V / sites_per_thread + 255) / 256;
    long cap = (long)ctx->num_sms * ctas_per_sm;
    return (int)std::max<long>(1, std::min(want, cap));
}

#define LQX_BY_KIND(KERNEL, T, kind, ...)                                                       \
    switch ((int)(kind)) {                                                                      \
        case LQX_COMPLEX: KERNEL<T, 2><<<grid, 256, 0, ctx->stream>>>(__VA_ARGS__); break;      \
        case LQX_COLORVEC: KERNEL<T, 6><<<grid, 256, 0, ctx->stream>>>(__VA_ARGS__); break;     \
        case LQX_COLORMAT: KERNEL<T, 18><<<grid, 256, 0, ctx->stream>>>(__VA_ARGS__); break;    \
        default: KERNEL<T, 24><<<grid, 256, 0, ctx->stream>>>(__VA_ARGS__); break;              \
    }

}  // namespace

// =============================================================================================
// C entry points
// =============================================================================================
extern "C" int lqx_copy(lqx_field* r, const lqx_field* a) { return flat_dispatch<0>(r, a, nullptr, 0.0); }
extern "C" int lqx_axpy(lqx_field* r, const lqx_field* s0, double kappa, const lqx_field* h) {
    return flat_dispatch<1>(r, s0, h, kappa);
}
extern "C" int lqx_scale(lqx_field* r, double s, const lqx_field* a) { return flat_dispatch<2>(r, a, nullptr, s); }
extern "C" int lqx_divide(lqx_field* r, const lqx_field* a, double nrm) { return flat_dispatch<3>(r, a, nullptr, nrm); }

extern "C" int lqx_shift(lqx_field* r, const lqx_field* a, lqx_dir dir, int mu) {
    lqx_ctx* ctx;
    int rc = check_same(&ctx, {r, a});
    if (rc) return rc;
    if (mu < 0 || mu > 3 || (dir != LQX_FORWARD && dir != LQX_BACKWARD)) return lqx_fail(ctx, LQX_EINVAL, "mu/dir");
    if (r->kind != a->kind) return lqx_fail(ctx, LQX_ETYPE, "shift: kinds differ");
    if (lqx_same(r, a)) return lqx_fail(ctx, LQX_EALIAS, "shift: in place");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    return r->prec == LQX_F32 ? shift_launch<float, false>(ctx, r, 0.0, nullptr, a, (int)dir, mu)
                              : shift_launch<double, false>(ctx, r, 0.0, nullptr, a, (int)dir, mu);
}

extern "C" int lqx_ax_minus_shift(lqx_field* r, double alpha, const lqx_field* a, const lqx_field* b, lqx_dir dir,
                                  int mu) {
    lqx_ctx* ctx;
    int rc = check_same(&ctx, {r, a, b});
    if (rc) return rc;
    if (mu < 0 || mu > 3 || (dir != LQX_FORWARD && dir != LQX_BACKWARD)) return lqx_fail(ctx, LQX_EINVAL, "mu/dir");
    if (r->kind != a->kind || r->kind != b->kind) return lqx_fail(ctx, LQX_ETYPE, "ax_minus_shift: kinds differ");
    if (lqx_same(r, b)) return lqx_fail(ctx, LQX_EALIAS, "ax_minus_shift: destination is the shifted operand");
    if (lqx_same(r, a) && !lqx_identical(r, a)) return lqx_fail(ctx, LQX_EALIAS, "ax_minus_shift: destination partially overlaps A");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    return r->prec == LQX_F32 ? shift_launch<float, true>(ctx, r, alpha, a, b, (int)dir, mu)
                              : shift_launch<double, true>(ctx, r, alpha, a, b, (int)dir, mu);
}

extern "C" int lqx_mm_plus_madj(lqx_field* r, const lqx_field* a, const lqx_field* b, const lqx_field* c,
                                const lqx_field* d) {
    lqx_ctx* ctx;
    int rc = check_same(&ctx, {r, a, b, c, d});
    if (rc) return rc;
    for (const lqx_field* f : {(const lqx_field*)r, a, b, c, d})
        if (f->kind != LQX_COLORMAT) return lqx_fail(ctx, LQX_ETYPE, "mm_plus_madj wants colour matrices");
    bool inplace = false;  // site-local: r may BE one of the operands (A21), never overlap one partially
    for (const lqx_field* f : {a, b, c, d}) {
        if (lqx_identical(r, f)) inplace = true;
        else if (lqx_same(r, f)) return lqx_fail(ctx, LQX_EALIAS, "mm_plus_madj: destination partially overlaps an operand");
    }
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const int V = ctx->geo.V, grid = (V + 127) / 128;
    LqxTimed timed(ctx, LQX_K_CATALOGUE);
#define LQX_FORM1(T, IP) k_mm_plus_madj<T, IP><<<grid, 128, 0, ctx->stream>>>(V, (const T*)a->data, (const T*)b->data, (const T*)c->data, (const T*)d->data, (T*)r->data)
    if (r->prec == LQX_F32) {
        if (inplace) LQX_FORM1(float, true);
        else LQX_FORM1(float, false);
    } else {
        if (inplace) LQX_FORM1(double, true);
        else LQX_FORM1(double, false);
    }
#undef LQX_FORM1
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}

extern "C" int lqx_trace_mm(lqx_field* c, const lqx_field* a, const lqx_field* b) {
    lqx_ctx* ctx;
    int rc = check_same(&ctx, {c, a, b});
    if (rc) return rc;
    if (c->kind != LQX_COMPLEX || a->kind != LQX_COLORMAT || b->kind != LQX_COLORMAT)
        return lqx_fail(ctx, LQX_ETYPE, "trace_mm: complex = trace(matrix*matrix)");
    if (lqx_same(c, a) || lqx_same(c, b)) return lqx_fail(ctx, LQX_EALIAS, "trace_mm: destination overlaps an operand");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const int V = ctx->geo.V, grid = (V + 127) / 128;
    LqxTimed timed(ctx, LQX_K_CATALOGUE);
    if (c->prec == LQX_F32)
        k_trace_mm<float><<<grid, 128, 0, ctx->stream>>>(V, (const float*)a->data, (const float*)b->data, (float*)c->data);
    else
        k_trace_mm<double><<<grid, 128, 0, ctx->stream>>>(V, (const double*)a->data, (const double*)b->data, (double*)c->data);
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}

extern "C" int lqx_mat_vec(lqx_field* w, const lqx_field* m, const lqx_field* v) {
    lqx_ctx* ctx;
    int rc = check_same(&ctx, {w, m, v});
    if (rc) return rc;
    if (m->kind != LQX_COLORMAT || w->kind != v->kind || (v->kind != LQX_COLORVEC && v->kind != LQX_FERMION))
        return lqx_fail(ctx, LQX_ETYPE, "mat_vec: matrix * (colour vector | fermion)");
    if (lqx_same(w, m) || (lqx_same(w, v) && !lqx_identical(w, v))) return lqx_fail(ctx, LQX_EALIAS, "mat_vec: destination overlaps an operand");
    const bool inplace = lqx_identical(w, v);  // v = M*v in place (A21)
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const int V = ctx->geo.V, grid = (V + 127) / 128;
    LqxTimed timed(ctx, LQX_K_CATALOGUE);
    const bool ferm = v->kind == LQX_FERMION;
#define LQX_FORM4(T, NS, IP) k_mat_vec<T, NS, IP><<<grid, 128, 0, ctx->stream>>>(V, (const T*)m->data, (const T*)v->data, (T*)w->data)
#define LQX_FORM4_T(T)                          \
    if (ferm) {                                 \
        if (inplace) LQX_FORM4(T, 4, true);     \
        else LQX_FORM4(T, 4, false);            \
    } else {                                    \
        if (inplace) LQX_FORM4(T, 1, true);     \
        else LQX_FORM4(T, 1, false);            \
    }
    if (w->prec == LQX_F32) {
        LQX_FORM4_T(float)
    } else {
        LQX_FORM4_T(double)
    }
#undef LQX_FORM4_T
#undef LQX_FORM4
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}

extern "C" int lqx_norm2(const lqx_field* f, double* out) {
    if (!f || !out) return LQX_EINVAL;
    lqx_ctx* ctx = f->ctx;
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const int grid = reduce_grid(ctx, 2);
    int rc = lqx_ensure_partials(ctx, (size_t)grid);
    if (rc) return rc;
    const int V = ctx->geo.V;
    {
        LqxTimed timed(ctx, LQX_K_REDUCE);
        if (f->prec == LQX_F32) {
            LQX_BY_KIND(k_norm2, float, f->kind, V, (const float*)f->data, ctx->d_partials, ctx->d_ticket, ctx->h_result)
        } else {
            LQX_BY_KIND(k_norm2, double, f->kind, V, (const double*)f->data, ctx->d_partials, ctx->d_ticket, ctx->h_result)
        }
    }
    LQX_LAUNCH_CHECK(ctx);
    return lqx_fetch_result(ctx, 1, out);
}

namespace {
// one wave of CTAs: a fixed function of the lattice and the SM count only (deterministic summation tree)
template <typename T, int NREAL, int SUB>
int sum_launch(lqx_ctx* ctx, const lqx_field* f) {
    constexpr int W = Vec128<T>::W, NQ = (NREAL + W - 1) / W, WARPS = NQ * SUB;
    const int nblk = ctx->geo.Vpad / 32;
    const int per_sm = std::max(1, std::min(32, 64 / WARPS));
    const int grid = (int)std::max<long>(1, std::min<long>((nblk + SUB - 1) / SUB, (long)ctx->num_sms * per_sm));
    int rc = lqx_ensure_partials(ctx, (size_t)grid * NREAL);
    if (rc) return rc;
    {
        LqxTimed timed(ctx, LQX_K_REDUCE);
        k_sum<T, NREAL, SUB><<<grid, 32 * WARPS, 0, ctx->stream>>>(nblk, (const T*)f->data, ctx->d_partials, ctx->d_ticket, ctx->h_result);
    }
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}
}  // namespace

extern "C" int lqx_sum(const lqx_field* f, double* out) {
    if (!f || !out) return LQX_EINVAL;
    lqx_ctx* ctx = f->ctx;
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const int nc = 2 * (int)f->kind;
    int rc;
    // SUB warps per chunk position, so that a CTA has 16-24 warps whatever the site object
    if (f->prec == LQX_F32) {
        switch ((int)f->kind) {
            case LQX_COMPLEX: rc = sum_launch<float, 2, 16>(ctx, f); break;
            case LQX_COLORVEC: rc = sum_launch<float, 6, 8>(ctx, f); break;
            case LQX_COLORMAT: rc = sum_launch<float, 18, 4>(ctx, f); break;
            default: rc = sum_launch<float, 24, 3>(ctx, f); break;
        }
    } else {
        switch ((int)f->kind) {
            case LQX_COMPLEX: rc = sum_launch<double, 2, 16>(ctx, f); break;
            case LQX_COLORVEC: rc = sum_launch<double, 6, 6>(ctx, f); break;
            case LQX_COLORMAT: rc = sum_launch<double, 18, 2>(ctx, f); break;
            default: rc = sum_launch<double, 24, 2>(ctx, f); break;
        }
    }
    if (rc) return rc;
    return lqx_fetch_result(ctx, nc, out);
}

extern "C" int lqx_trace(const lqx_field* m, double out[2]) {
    if (!m || !out) return LQX_EINVAL;
    lqx_ctx* ctx = m->ctx;
    if (m->kind != LQX_COLORMAT) return lqx_fail(ctx, LQX_ETYPE, "trace wants a colour matrix");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const int grid = reduce_grid(ctx, 2);
    int rc = lqx_ensure_partials(ctx, (size_t)grid * 2);
    if (rc) return rc;
    const int V = ctx->geo.V;
    {
        LqxTimed timed(ctx, LQX_K_REDUCE);
        if (m->prec == LQX_F32) k_trace<float><<<grid, 256, 0, ctx->stream>>>(V, (const float*)m->data, ctx->d_partials, ctx->d_ticket, ctx->h_result);
        else k_trace<double><<<grid, 256, 0, ctx->stream>>>(V, (const double*)m->data, ctx->d_partials, ctx->d_ticket, ctx->h_result);
    }
    LQX_LAUNCH_CHECK(ctx);
    return lqx_fetch_result(ctx, 2, out);
}
