// lqx expression catalogue and standalone global reductions (a9).
// Every entry point is one pass over HBM: the whole expression, shift included, is evaluated per
// site with no temporaries (the paper's evaluate()), operands read from the
// site-fastest SoA planes so that a warp touches 32 consecutive reals of each plane.
#include "lqx_internal.cuh"

namespace {

// NS consecutive sites of one plane as one 8/16-byte access
template <typename T, int NS>
struct alignas(sizeof(T) * NS) Pack {
    T v[NS];
};
template <typename T>
struct VecWidth {
    static constexpr int value = 16 / sizeof(T);  // 128-bit accesses
};

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
// flat elementwise kernels over the whole plane array (pad included: it is never read for results)
// mode 0: r = a ; 1: r = a + k*b ; 2: r = k*a ; 3: r = a / k
// ---------------------------------------------------------------------------------------------
template <typename T, int MODE>
__global__ void k_flat(size_t nvec, T k, const T* __restrict__ a, const T* __restrict__ b, T* __restrict__ r) {
    constexpr int W = VecWidth<T>::value;
    typedef Pack<T, W> P;
    const size_t step = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += step) {
        P va = reinterpret_cast<const P*>(a)[i];
        P vb;
        if (MODE == 1) vb = reinterpret_cast<const P*>(b)[i];
        P vr;
#pragma unroll
        for (int j = 0; j < W; ++j) {
            if (MODE == 0) vr.v[j] = va.v[j];
            if (MODE == 1) vr.v[j] = fma(k, vb.v[j], va.v[j]);
            if (MODE == 2) vr.v[j] = k * va.v[j];
            if (MODE == 3) vr.v[j] = va.v[j] / k;
        }
        reinterpret_cast<P*>(r)[i] = vr;
    }
}

template <typename T, int MODE>
int flat_launch(lqx_ctx* ctx, lqx_field* r, const lqx_field* a, const lqx_field* b, double k) {
    const size_t n = (size_t)ctx->geo.stride * 2 * (int)r->kind;
    const size_t nvec = n / VecWidth<T>::value;
    const int block = 256;
    size_t want = (nvec + block - 1) / block;
    int grid = (int)std::min<size_t>(want, (size_t)ctx->num_sms * 16);
    if (grid < 1) grid = 1;
    LqxTimed timed(ctx, LQX_K_CATALOGUE);
    k_flat<T, MODE><<<grid, block, 0, ctx->stream>>>(nvec, (T)k, (const T*)a->data, b ? (const T*)b->data : nullptr,
                                                      (T*)r->data);
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}

template <int MODE>
int flat_dispatch(lqx_field* r, const lqx_field* a, const lqx_field* b, double k) {
    lqx_ctx* ctx;
    int rc = b ? check_same(&ctx, {r, a, b}) : check_same(&ctx, {r, a});
    if (rc) return rc;
    if (r->kind != a->kind || (b && b->kind != a->kind)) return lqx_fail(ctx, LQX_ETYPE, "field kinds differ");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    return r->prec == LQX_F32 ? flat_launch<float, MODE>(ctx, r, a, b, k) : flat_launch<double, MODE>(ctx, r, a, b, k);
}

// ---------------------------------------------------------------------------------------------
// shift and form (iii): one thread = NS consecutive sites of one plane (blockIdx.y = plane).
// For mu >= 1 the neighbours of NS aligned consecutive sites are NS aligned consecutive sites
// (L0 % NS == 0), so the shifted operand is one vector access; for mu == 0 they straddle the
// vector boundary and wrap at the row end, so they are read element-wise (L1 serves the overlap).
// AX = false: r = shift(b);  AX = true: r = alpha*a - shift(b)
// ---------------------------------------------------------------------------------------------
template <typename T, int NS, bool AX>
__global__ void k_shift(const __grid_constant__ Geo g, int dir, int mu, T alpha, const T* __restrict__ a, const T* __restrict__ b,
                        T* __restrict__ r) {
    typedef Pack<T, NS> P;
    const int s0 = (blockIdx.x * blockDim.x + threadIdx.x) * NS;
    if (s0 >= g.V) return;
    const size_t plane = (size_t)blockIdx.y * g.stride;
    int x[4];
    site_coords(g, s0, x);
    P vb;
    if (mu == 0 && NS > 1) {
#pragma unroll
        for (int j = 0; j < NS; ++j) {
            int xj = x[0] + j + dir;
            xj = xj < 0 ? xj + g.L[0] : (xj >= g.L[0] ? xj - g.L[0] : xj);
            vb.v[j] = __ldg(b + plane + (s0 - x[0]) + xj);
        }
    } else {
        const int n0 = dir > 0 ? nbr_fwd(g, s0, x, mu) : nbr_bwd(g, s0, x, mu);
        vb = *reinterpret_cast<const P*>(b + plane + n0);
    }
    P vr;
    if (AX) {
        P va = *reinterpret_cast<const P*>(a + plane + s0);
#pragma unroll
        for (int j = 0; j < NS; ++j) vr.v[j] = mul_rn(alpha, va.v[j]) - vb.v[j];  // alpha*A rounded once, as written
    } else {
        vr = vb;
    }
    *reinterpret_cast<P*>(r + plane + s0) = vr;
}

template <typename T, bool AX>
int shift_launch(lqx_ctx* ctx, lqx_field* r, double alpha, const lqx_field* a, const lqx_field* b, int dir, int mu) {
    const Geo& g = ctx->geo;
    constexpr int W = VecWidth<T>::value;
    const int nplanes = 2 * (int)r->kind;
    const int block = 256;
    const T* pa = a ? (const T*)a->data : nullptr;
    LqxTimed timed(ctx, LQX_K_CATALOGUE);
    if (g.L[0] % W == 0) {
        dim3 grid((g.V / W + block - 1) / block, nplanes);
        k_shift<T, W, AX><<<grid, block, 0, ctx->stream>>>(g, dir, mu, (T)alpha, pa, (const T*)b->data, (T*)r->data);
    } else {
        dim3 grid((g.V + block - 1) / block, nplanes);
        k_shift<T, 1, AX><<<grid, block, 0, ctx->stream>>>(g, dir, mu, (T)alpha, pa, (const T*)b->data, (T*)r->data);
    }
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}

// ---------------------------------------------------------------------------------------------
// site-local matrix forms: one thread per site, all operands of the site in registers
// ---------------------------------------------------------------------------------------------
// form (i) R = A*B + C*adj(D)
template <typename T>
__global__ void __launch_bounds__(128) k_mm_plus_madj(const __grid_constant__ Geo g, const T* __restrict__ a, const T* __restrict__ b,
                                                      const T* __restrict__ c, const T* __restrict__ d,
                                                      T* __restrict__ r) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.V) return;
    Mat3<T> ma = load_mat(a, g.stride, s), mb = load_mat(b, g.stride, s);
    Mat3<T> mc = load_mat(c, g.stride, s), md = load_mat(d, g.stride, s);
    Mat3<T> acc = mul_nn(ma, mb);
    mac_na(acc, mc, md);
    store_mat(r, g.stride, s, acc);
}
// form (ii) c = trace(A*B) = sum_ik A_ik B_ki
template <typename T>
__global__ void __launch_bounds__(128) k_trace_mm(const __grid_constant__ Geo g, const T* __restrict__ a, const T* __restrict__ b,
                                                  T* __restrict__ c) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.V) return;
    Mat3<T> ma = load_mat(a, g.stride, s), mb = load_mat(b, g.stride, s);
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
    c[s] = re;
    c[(size_t)g.stride + s] = im;
}
// form (iv) w = M*v per spin component
template <typename T, int NSPIN>
__global__ void __launch_bounds__(128) k_mat_vec(const __grid_constant__ Geo g, const T* __restrict__ m, const T* __restrict__ v,
                                                 T* __restrict__ w) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.V) return;
    Mat3<T> mm = load_mat(m, g.stride, s);
#pragma unroll
    for (int a = 0; a < NSPIN; ++a) {
        Vec3<T> vv = load_vec(v, g.stride, s, a);
        Vec3<T> ww;
#pragma unroll
        for (int i = 0; i < 3; ++i) ww.re[i] = ww.im[i] = T(0);
        mac_mv(ww, mm, vv);
        store_vec(w, g.stride, s, a, ww);
    }
}

// ---------------------------------------------------------------------------------------------
// standalone reductions: fp64 accumulation per thread over a grid-stride loop with a FIXED grid,
// then the deterministic block tree (lqx_internal.cuh) and the second stage (lqx_core.cu).
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void k_norm2(const __grid_constant__ Geo g, int nplanes, const T* __restrict__ f, double* __restrict__ partials) {
    constexpr int W = VecWidth<T>::value;
    typedef Pack<T, W> P;
    double acc[1] = {0.0};
    const int nv = g.V / W;  // full vectors per plane
    const int step = gridDim.x * blockDim.x;
    for (int p = 0; p < nplanes; ++p) {
        const T* base = f + (size_t)p * g.stride;
        for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nv; i += step) {
            P v = reinterpret_cast<const P*>(base)[i];
#pragma unroll
            for (int j = 0; j < W; ++j) acc[0] = fma((double)v.v[j], (double)v.v[j], acc[0]);
        }
        for (int i = nv * W + blockIdx.x * blockDim.x + threadIdx.x; i < g.V; i += step) {
            double t = (double)base[i];
            acc[0] = fma(t, t, acc[0]);
        }
    }
    block_reduce_store<1>(acc, partials, gridDim.x, blockIdx.x);
}
// sum over sites of every plane -> NC = nplanes doubles
template <typename T, int NC>
__global__ void k_sum(const __grid_constant__ Geo g, const T* __restrict__ f, double* __restrict__ partials) {
    double acc[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) acc[c] = 0.0;
    const int step = gridDim.x * blockDim.x;
    for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < g.V; s += step) {
#pragma unroll
        for (int c = 0; c < NC; ++c) acc[c] += (double)__ldg(f + (size_t)c * g.stride + s);
    }
    block_reduce_store<NC>(acc, partials, gridDim.x, blockIdx.x);
}
// sum_x tr M(x): planes of the diagonal elements (0,0),(1,1),(2,2)
template <typename T>
__global__ void k_trace(const __grid_constant__ Geo g, const T* __restrict__ m, double* __restrict__ partials) {
    double acc[2] = {0.0, 0.0};
    const int step = gridDim.x * blockDim.x;
    for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < g.V; s += step) {
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            acc[0] += (double)__ldg(m + (size_t)(2 * (4 * i)) * g.stride + s);
            acc[1] += (double)__ldg(m + (size_t)(2 * (4 * i) + 1) * g.stride + s);
        }
    }
    block_reduce_store<2>(acc, partials, gridDim.x, blockIdx.x);
}

int reduce_grid(const lqx_ctx* ctx, int per_thread_items) {
    // fixed function of V only => deterministic summation tree
    long want = ((long)ctx->geo.V / per_thread_items + 255) / 256;
    long cap = (long)ctx->num_sms * 8;
    return (int)std::max<long>(1, std::min(want, cap));
}

template <typename T>
int sum_launch(lqx_ctx* ctx, const lqx_field* f, int grid) {
    const T* p = (const T*)f->data;
    switch ((int)f->kind) {
        case LQX_COMPLEX: k_sum<T, 2><<<grid, 256, 0, ctx->stream>>>(ctx->geo, p, ctx->d_partials); break;
        case LQX_COLORVEC: k_sum<T, 6><<<grid, 256, 0, ctx->stream>>>(ctx->geo, p, ctx->d_partials); break;
        case LQX_COLORMAT: k_sum<T, 18><<<grid, 256, 0, ctx->stream>>>(ctx->geo, p, ctx->d_partials); break;
        default: k_sum<T, 24><<<grid, 256, 0, ctx->stream>>>(ctx->geo, p, ctx->d_partials); break;
    }
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
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
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const Geo& g = ctx->geo;
    const int grid = (g.V + 127) / 128;
    LqxTimed timed(ctx, LQX_K_CATALOGUE);
    if (r->prec == LQX_F32)
        k_mm_plus_madj<float><<<grid, 128, 0, ctx->stream>>>(g, (const float*)a->data, (const float*)b->data,
                                                            (const float*)c->data, (const float*)d->data, (float*)r->data);
    else
        k_mm_plus_madj<double><<<grid, 128, 0, ctx->stream>>>(g, (const double*)a->data, (const double*)b->data,
                                                             (const double*)c->data, (const double*)d->data, (double*)r->data);
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}

extern "C" int lqx_trace_mm(lqx_field* c, const lqx_field* a, const lqx_field* b) {
    lqx_ctx* ctx;
    int rc = check_same(&ctx, {c, a, b});
    if (rc) return rc;
    if (c->kind != LQX_COMPLEX || a->kind != LQX_COLORMAT || b->kind != LQX_COLORMAT)
        return lqx_fail(ctx, LQX_ETYPE, "trace_mm: complex = trace(matrix*matrix)");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const Geo& g = ctx->geo;
    const int grid = (g.V + 127) / 128;
    LqxTimed timed(ctx, LQX_K_CATALOGUE);
    if (c->prec == LQX_F32)
        k_trace_mm<float><<<grid, 128, 0, ctx->stream>>>(g, (const float*)a->data, (const float*)b->data, (float*)c->data);
    else
        k_trace_mm<double><<<grid, 128, 0, ctx->stream>>>(g, (const double*)a->data, (const double*)b->data, (double*)c->data);
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}

extern "C" int lqx_mat_vec(lqx_field* w, const lqx_field* m, const lqx_field* v) {
    lqx_ctx* ctx;
    int rc = check_same(&ctx, {w, m, v});
    if (rc) return rc;
    if (m->kind != LQX_COLORMAT || w->kind != v->kind || (v->kind != LQX_COLORVEC && v->kind != LQX_FERMION))
        return lqx_fail(ctx, LQX_ETYPE, "mat_vec: matrix * (colour vector | fermion)");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const Geo& g = ctx->geo;
    const int grid = (g.V + 127) / 128;
    LqxTimed timed(ctx, LQX_K_CATALOGUE);
    const bool ferm = v->kind == LQX_FERMION;
    if (w->prec == LQX_F32) {
        if (ferm) k_mat_vec<float, 4><<<grid, 128, 0, ctx->stream>>>(g, (const float*)m->data, (const float*)v->data, (float*)w->data);
        else k_mat_vec<float, 1><<<grid, 128, 0, ctx->stream>>>(g, (const float*)m->data, (const float*)v->data, (float*)w->data);
    } else {
        if (ferm) k_mat_vec<double, 4><<<grid, 128, 0, ctx->stream>>>(g, (const double*)m->data, (const double*)v->data, (double*)w->data);
        else k_mat_vec<double, 1><<<grid, 128, 0, ctx->stream>>>(g, (const double*)m->data, (const double*)v->data, (double*)w->data);
    }
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}

extern "C" int lqx_norm2(const lqx_field* f, double* out) {
    if (!f || !out) return LQX_EINVAL;
    lqx_ctx* ctx = f->ctx;
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const int grid = reduce_grid(ctx, 8);
    int rc = lqx_ensure_partials(ctx, (size_t)grid);
    if (rc) return rc;
    {
        LqxTimed timed(ctx, LQX_K_REDUCE);
        if (f->prec == LQX_F32) k_norm2<float><<<grid, 256, 0, ctx->stream>>>(ctx->geo, 2 * (int)f->kind, (const float*)f->data, ctx->d_partials);
        else k_norm2<double><<<grid, 256, 0, ctx->stream>>>(ctx->geo, 2 * (int)f->kind, (const double*)f->data, ctx->d_partials);
    }
    LQX_LAUNCH_CHECK(ctx);
    rc = lqx_reduce_finish(ctx, grid, 1, ctx->d_result);
    if (rc) return rc;
    return lqx_fetch_result(ctx, 1, out);
}

extern "C" int lqx_sum(const lqx_field* f, double* out) {
    if (!f || !out) return LQX_EINVAL;
    lqx_ctx* ctx = f->ctx;
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const int nc = 2 * (int)f->kind;
    const int grid = reduce_grid(ctx, 4);
    int rc = lqx_ensure_partials(ctx, (size_t)grid * nc);
    if (rc) return rc;
    {
        LqxTimed timed(ctx, LQX_K_REDUCE);
        rc = f->prec == LQX_F32 ? sum_launch<float>(ctx, f, grid) : sum_launch<double>(ctx, f, grid);
    }
    if (rc) return rc;
    rc = lqx_reduce_finish(ctx, grid, nc, ctx->d_result);
    if (rc) return rc;
    return lqx_fetch_result(ctx, nc, out);
}

extern "C" int lqx_trace(const lqx_field* m, double out[2]) {
    if (!m || !out) return LQX_EINVAL;
    lqx_ctx* ctx = m->ctx;
    if (m->kind != LQX_COLORMAT) return lqx_fail(ctx, LQX_ETYPE, "trace wants a colour matrix");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const int grid = reduce_grid(ctx, 4);
    int rc = lqx_ensure_partials(ctx, (size_t)grid * 2);
    if (rc) return rc;
    {
        LqxTimed timed(ctx, LQX_K_REDUCE);
        if (m->prec == LQX_F32) k_trace<float><<<grid, 256, 0, ctx->stream>>>(ctx->geo, (const float*)m->data, ctx->d_partials);
        else k_trace<double><<<grid, 256, 0, ctx->stream>>>(ctx->geo, (const double*)m->data, ctx->d_partials);
    }
    LQX_LAUNCH_CHECK(ctx);
    rc = lqx_reduce_finish(ctx, grid, 2, ctx->d_result);
    if (rc) return rc;
    return lqx_fetch_result(ctx, 2, out);
}
