// lqx core: context, geometry, device field store with QDP-order <-> blocked-SoA converters
// (SURVEY 8(a) a1, a2; PAPER.md:101-103 site tables, :195-202 push/pop/free), error handling and
// the result hand-off of the reductions.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "lqx_internal.cuh"

// --------------------------------------------------------------------------------------------
// errors
// --------------------------------------------------------------------------------------------
int lqx_fail(lqx_ctx* ctx, int code, const char* what) {
    if (ctx) ctx->last_error = what ? what : "";
    return code;
}
int lqx_cuda_fail(lqx_ctx* ctx, cudaError_t e, const char* where) {
    if (ctx) {
        ctx->last_error = std::string(where ? where : "cuda") + ": " + cudaGetErrorString(e);
    }
    return LQX_ECUDA;
}

extern "C" const char* lqx_strerror(int code) {
    switch (code) {
        case LQX_OK: return "ok";
        case LQX_EINVAL: return "invalid argument";
        case LQX_ETYPE: return "operand kind or precision mismatch";
        case LQX_EGEOM: return "geometry mismatch or unsupported lattice";
        case LQX_EALIAS: return "destination aliases a shifted operand";
        case LQX_ECUDA: return "CUDA error";
        case LQX_ENOMEM: return "out of memory";
        default: return "unknown lqx status";
    }
}
extern "C" const char* lqx_last_error(const lqx_ctx* ctx) { return ctx ? ctx->last_error.c_str() : ""; }
extern "C" const char* lqx_version(void) { return "lqx 0.1 (sm_100a)"; }

// --------------------------------------------------------------------------------------------
// geometry
// --------------------------------------------------------------------------------------------
static FastDiv make_fastdiv(uint32_t d) {
    FastDiv f;
    f.d = d;
    uint32_t sh = 0;
    while ((1ull << sh) < d) ++sh;
    f.sh = sh;
    unsigned __int128 num = (unsigned __int128)1 << (31 + sh);
    f.mul = (uint32_t)((num + d - 1) / d);
    return f;
}

extern "C" int lqx_init(const int dims[4], int device, void* cuda_stream, lqx_ctx** out) {
    if (!dims || !out) return LQX_EINVAL;
    *out = nullptr;
    int64_t v = 1;
    for (int d = 0; d < 4; ++d) {
        if (dims[d] < 1) return LQX_EGEOM;
        v *= dims[d];
        if (v >= ((int64_t)1 << 31) - 64) return LQX_EGEOM;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return LQX_ECUDA;
    if (cudaSetDevice(device) != cudaSuccess) return LQX_ECUDA;
    lqx_ctx* c = new (std::nothrow) lqx_ctx();
    if (!c) return LQX_ENOMEM;
    Geo& g = c->geo;
    int st = 1;
    for (int d = 0; d < 4; ++d) {
        g.L[d] = dims[d];
        g.stride_site[d] = st;
        st *= dims[d];
    }
    g.V = (int)v;
    g.Vpad = (int)((v + 31) & ~(int64_t)31);
    g.d0 = make_fastdiv((uint32_t)dims[0]);
    g.d1 = make_fastdiv((uint32_t)dims[1]);
    g.d2 = make_fastdiv((uint32_t)dims[2]);
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    c->d_partials = nullptr;
    c->partials_cap = 0;
    c->d_result = nullptr;
    c->h_result = nullptr;
    c->launches = 0;
    c->opt_smear_variant = 0;
    c->opt_plaq_variant = 0;
    c->opt_block = 0;
    c->opt_hop_block = 0;
    for (int p = 0; p < 2; ++p) {
        c->tuned_smear_variant[p] = 0, c->tuned_smear_tile[p] = -1, c->tuned_plaq_variant[p] = 0;
        c->tuned_hop_block[p] = 0, c->tuned_jacobi_block[p] = 0, c->tuned_jacobi_sites[p] = 0;
    }
    c->last_smear_variant = 0, c->last_smear_lane_ops = 0, c->last_smear_kernel = "";
    c->opt_tile = -1;
    c->opt_bulk_fill = 0;
    c->opt_jacobi_block = c->opt_jacobi_sites = 0;
    c->timing = false;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) {
        delete c;
        return LQX_ECUDA;
    }
    c->num_sms = prop.multiProcessorCount;
    c->d_ticket = nullptr;
    c->stage = nullptr;
    for (int k = 0; k < 12; ++k) c->host_work[k] = nullptr;
    c->pipe_stream[0] = c->pipe_stream[1] = nullptr;
    c->opt_host_slabs = -1;
    c->stage_cap = 0;
    if (cudaMalloc(&c->d_result, 64 * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&c->d_ticket, sizeof(unsigned int)) != cudaSuccess ||
        cudaHostAlloc(&c->h_result, 64 * sizeof(double), cudaHostAllocPortable | cudaHostAllocMapped) != cudaSuccess ||
        cudaMemset(c->d_ticket, 0, sizeof(unsigned int)) != cudaSuccess) {
        if (c->d_result) cudaFree(c->d_result);
        if (c->d_ticket) cudaFree(c->d_ticket);
        cudaGetLastError();
        delete c;
        return LQX_ENOMEM;
    }
    *out = c;
    return LQX_OK;
}

extern "C" int lqx_finalize(lqx_ctx* ctx) {
    if (!ctx) return LQX_EINVAL;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    lqx_jit_release(ctx);
    lqx_staged_release(ctx);
    for (lqx_field* f : ctx->fields) {
        if (f->owned && f->data) cudaFree(f->data);
        delete f;
    }
    for (auto& v : ctx->timers)
        for (auto& pr : v) {
            cudaEventDestroy(pr.first);
            cudaEventDestroy(pr.second);
        }
    for (cudaEvent_t e : ctx->pipe_events) cudaEventDestroy(e);
    for (int k = 0; k < 2; ++k)
        if (ctx->pipe_stream[k]) cudaStreamDestroy(ctx->pipe_stream[k]);
    if (ctx->d_partials) cudaFree(ctx->d_partials);
    if (ctx->stage) cudaFree(ctx->stage);
    if (ctx->d_result) cudaFree(ctx->d_result);
    if (ctx->d_ticket) cudaFree(ctx->d_ticket);
    if (ctx->h_result) cudaFreeHost(ctx->h_result);
    delete ctx;
    return LQX_OK;
}

extern "C" int lqx_set_stream(lqx_ctx* ctx, void* cuda_stream) {
    if (!ctx) return LQX_EINVAL;
    // the context's scratch (reduction partials, staging buffer, pinned results) is ordered by its stream:
    // drain the old one before work is enqueued on the new one
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    LQX_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->stream = (cudaStream_t)cuda_stream;
    return LQX_OK;
}
extern "C" int64_t lqx_volume(const lqx_ctx* ctx) { return ctx ? ctx->geo.V : (int64_t)LQX_EINVAL; }
extern "C" int64_t lqx_padded_volume(const lqx_ctx* ctx) { return ctx ? ctx->geo.Vpad : (int64_t)LQX_EINVAL; }
extern "C" int64_t lqx_launch_count(const lqx_ctx* ctx) { return ctx ? ctx->launches : (int64_t)LQX_EINVAL; }
extern "C" int lqx_smear_info(const lqx_ctx* ctx, int* variant, int* lane_ops_per_site, char* kernel_name, int name_len) {
    if (!ctx) return LQX_EINVAL;
    if (variant) *variant = ctx->last_smear_variant;
    if (lane_ops_per_site) *lane_ops_per_site = ctx->last_smear_lane_ops;
    if (kernel_name && name_len > 0) {
        strncpy(kernel_name, ctx->last_smear_kernel ? ctx->last_smear_kernel : "", (size_t)name_len - 1);
        kernel_name[name_len - 1] = '\0';
    }
    return LQX_OK;
}

static bool valid_kind(int k) { return k == LQX_COMPLEX || k == LQX_COLORVEC || k == LQX_COLORMAT || k == LQX_FERMION; }
static bool valid_prec(int p) { return p == LQX_F32 || p == LQX_F64; }

extern "C" int64_t lqx_field_bytes(const lqx_ctx* ctx, lqx_kind kind, lqx_prec prec) {
    if (!ctx || !valid_kind(kind) || !valid_prec(prec)) return LQX_EINVAL;
    return (int64_t)ctx->geo.Vpad * 2 * (int)kind * (int)prec;
}

extern "C" int64_t lqx_field_offset(const lqx_ctx* ctx, lqx_kind kind, lqx_prec prec, int64_t site, int real_index) {
    if (!ctx || !valid_kind(kind) || !valid_prec(prec)) return LQX_EINVAL;
    const int nreal = 2 * (int)kind;
    if (site < 0 || site >= ctx->geo.V || real_index < 0 || real_index >= nreal) return LQX_EINVAL;
    return (int64_t)lqx_layout_offset((int)site, real_index, nreal, 16 / (int)prec);
}

extern "C" int lqx_set_option(lqx_ctx* ctx, const char* key, int value) {
    if (!ctx || !key) return LQX_EINVAL;
    if (!strcmp(key, "smear_variant")) ctx->opt_smear_variant = value;
    else if (!strcmp(key, "plaq_variant")) ctx->opt_plaq_variant = value;
    else if (!strcmp(key, "block")) ctx->opt_block = value;
    else if (!strcmp(key, "hop_block")) ctx->opt_hop_block = value;
    else if (!strcmp(key, "tile")) ctx->opt_tile = value;
    else if (!strcmp(key, "bulk_fill")) ctx->opt_bulk_fill = value;
    else if (!strcmp(key, "jacobi_block")) ctx->opt_jacobi_block = value;
    else if (!strcmp(key, "jacobi_sites")) ctx->opt_jacobi_sites = value;
    else if (!strcmp(key, "time_kernels")) ctx->timing = value != 0;
    else if (!strcmp(key, "host_slabs")) ctx->opt_host_slabs = value;
    else return lqx_fail(ctx, LQX_EINVAL, "unknown option");
    return LQX_OK;
}

extern "C" int lqx_kernel_time(lqx_ctx* ctx, int which, double* total_ms, int* count) {
    if (!ctx || which < 0 || which >= LQX_NUM_KERNEL_CLASSES || !total_ms || !count) return LQX_EINVAL;
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    LQX_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    double tot = 0.0;
    int n = 0;
    for (auto& pr : ctx->timers[which]) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, pr.first, pr.second) == cudaSuccess) {
            tot += ms;
            ++n;
        }
        cudaEventDestroy(pr.first);
        cudaEventDestroy(pr.second);
    }
    ctx->timers[which].clear();
    cudaGetLastError();
    *total_ms = tot;
    *count = n;
    return LQX_OK;
}

__global__ void k_neighbor_table(const __grid_constant__ Geo g, int dir, int mu, int32_t* __restrict__ out) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.V) return;
    int x[4];
    site_coords(g, s, x);
    out[s] = dir > 0 ? nbr_fwd(g, s, x, mu) : nbr_bwd(g, s, x, mu);
}

extern "C" int lqx_neighbor_table(lqx_ctx* ctx, lqx_dir dir, int mu, int32_t* host_out) {
    if (!ctx || !host_out) return LQX_EINVAL;
    if (mu < 0 || mu > 3 || (dir != LQX_FORWARD && dir != LQX_BACKWARD)) return lqx_fail(ctx, LQX_EINVAL, "mu/dir");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    int32_t* d = nullptr;
    const int V = ctx->geo.V;
    if (cudaMalloc(&d, (size_t)V * sizeof(int32_t)) != cudaSuccess) return lqx_fail(ctx, LQX_ENOMEM, "neighbor table");
    k_neighbor_table<<<(V + 255) / 256, 256, 0, ctx->stream>>>(ctx->geo, (int)dir, mu, d);
    ctx->launches++;
    cudaError_t e = cudaMemcpyAsync(host_out, d, (size_t)V * sizeof(int32_t), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(d);
    if (e != cudaSuccess) return lqx_cuda_fail(ctx, e, "neighbor table");
    return LQX_OK;
}

// --------------------------------------------------------------------------------------------
// fields
// --------------------------------------------------------------------------------------------
static int new_field(lqx_ctx* ctx, lqx_kind kind, lqx_prec prec, void* ptr, bool owned, lqx_field** out) {
    lqx_field* f = new (std::nothrow) lqx_field();
    if (!f) return lqx_fail(ctx, LQX_ENOMEM, "field handle");
    f->ctx = ctx;
    f->kind = kind;
    f->prec = prec;
    f->data = ptr;
    f->owned = owned;
    ctx->fields.push_back(f);
    *out = f;
    return LQX_OK;
}

extern "C" int lqx_field_alloc(lqx_ctx* ctx, lqx_kind kind, lqx_prec prec, lqx_field** out) {
    if (!ctx || !out) return LQX_EINVAL;
    *out = nullptr;
    if (!valid_kind(kind) || !valid_prec(prec)) return lqx_fail(ctx, LQX_EINVAL, "kind/prec");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    void* p = nullptr;
    size_t bytes = (size_t)lqx_field_bytes(ctx, kind, prec);
    if (cudaMalloc(&p, bytes) != cudaSuccess) {
        cudaGetLastError();
        return lqx_fail(ctx, LQX_ENOMEM, "cudaMalloc field");
    }
    // the pad lanes of the last 32-site block are never read for results, but keep them defined
    cudaError_t e = cudaMemsetAsync(p, 0, bytes, ctx->stream);
    if (e != cudaSuccess) {
        cudaFree(p);
        return lqx_cuda_fail(ctx, e, "memset");
    }
    int rc = new_field(ctx, kind, prec, p, true, out);
    if (rc != LQX_OK) cudaFree(p);
    return rc;
}

extern "C" int lqx_field_attach(lqx_ctx* ctx, lqx_kind kind, lqx_prec prec, void* dev_ptr, size_t bytes,
                                lqx_field** out) {
    if (!ctx || !out || !dev_ptr) return LQX_EINVAL;
    *out = nullptr;
    if (!valid_kind(kind) || !valid_prec(prec)) return lqx_fail(ctx, LQX_EINVAL, "kind/prec");
    if ((int64_t)bytes < lqx_field_bytes(ctx, kind, prec)) return lqx_fail(ctx, LQX_EINVAL, "attached buffer too small");
    if (((uintptr_t)dev_ptr & 255) != 0) return lqx_fail(ctx, LQX_EINVAL, "attached buffer not 256-byte aligned");
    return new_field(ctx, kind, prec, dev_ptr, false, out);
}

extern "C" int lqx_field_free(lqx_field* f) {
    if (!f) return LQX_EINVAL;
    lqx_ctx* ctx = f->ctx;
    auto it = std::find(ctx->fields.begin(), ctx->fields.end(), f);
    if (it == ctx->fields.end()) return lqx_fail(ctx, LQX_EINVAL, "unknown field handle");
    ctx->fields.erase(it);
    if (f->owned && f->data) {
        cudaSetDevice(ctx->device);
        cudaStreamSynchronize(ctx->stream);
        cudaFree(f->data);
    }
    delete f;
    return LQX_OK;
}
extern "C" void* lqx_field_data(const lqx_field* f) { return f ? f->data : nullptr; }
extern "C" int lqx_field_kind(const lqx_field* f) { return f ? (int)f->kind : LQX_EINVAL; }
extern "C" int lqx_field_prec(const lqx_field* f) { return f ? (int)f->prec : LQX_EINVAL; }

// AoS (QDP order) <-> blocked SoA.  Both sides of a 32-site layout block are the same 32*NREAL contiguous
// reals, so the conversion is a permutation staged through shared memory.  One CTA converts kTransposeBlocks
// consecutive layout blocks with 128-bit global accesses on both sides (a block starts on a 16-byte boundary
// in either order); NREAL is a template parameter so that the index arithmetic divides by constants -- with
// run-time divisors and 4-byte accesses the kernel was instruction-bound at 2.2 TB/s.  The last block of a
// lattice whose volume is not a multiple of 32 takes the element-wise path on its QDP-order side.
static const int kTransposeBlocks = 4;

template <typename T, int NREAL, bool TO_SOA>
__global__ void __launch_bounds__(256) k_transpose(int V, int blk0, int blk_end, const T* __restrict__ src, T* __restrict__ dst) {
    typedef typename Vec128<T>::type VT;
    constexpr int W = Vec128<T>::W, PITCH = NREAL + 1, NFULL = NREAL / W, REM = NREAL - NFULL * W, REMD = REM ? REM : 1;
    constexpr int E = 32 * NREAL, EV = E / W;  // reals and 128-bit vectors per block
    __shared__ T tiles[kTransposeBlocks][32 * PITCH];  // [block][local site][real], QDP order, padded pitch
    const int first = blk0 + blockIdx.x * kTransposeBlocks;
    const int nb = min(kTransposeBlocks, blk_end - first);
    // (local site, real) of element e of vector vi: QDP-order side / blocked side
    auto aos_pos = [](int vi, int e, int& ls, int& r) {
        const int idx = vi * W + e;
        ls = idx / NREAL;
        r = idx - ls * NREAL;
    };
    auto soa_pos = [](int vi, int e, int& ls, int& r) {
        if (vi < NFULL * 32) {
            ls = vi & 31;
            r = (vi >> 5) * W + e;
        } else {
            const int t = (vi - NFULL * 32) * W + e;
            ls = t / REMD;
            r = NFULL * W + (t - ls * REMD);
        }
    };
    for (int v = threadIdx.x; v < nb * EV; v += 256) {
        const int b = v / EV, vi = v - b * EV, blkid = first + b;
        const int ns = min(32, V - blkid * 32);
        const T* sp = src + (size_t)blkid * E;
        T* tile = tiles[b];
        if (ns == 32 || !TO_SOA) {  // the blocked side is padded to whole blocks
            T x[W];
            unpack(*reinterpret_cast<const VT*>(sp + vi * W), x);
#pragma unroll
            for (int e = 0; e < W; ++e) {
                int ls, r;
                if (TO_SOA) aos_pos(vi, e, ls, r);
                else soa_pos(vi, e, ls, r);
                tile[ls * PITCH + r] = x[e];
            }
        } else {
#pragma unroll
            for (int e = 0; e < W; ++e) {
                int ls, r;
                aos_pos(vi, e, ls, r);
                if (ls < ns) tile[ls * PITCH + r] = sp[vi * W + e];
            }
        }
    }
    __syncthreads();
    for (int v = threadIdx.x; v < nb * EV; v += 256) {
        const int b = v / EV, vi = v - b * EV, blkid = first + b;
        const int ns = min(32, V - blkid * 32);
        T* dp = dst + (size_t)blkid * E;
        const T* tile = tiles[b];
        if (TO_SOA) {
            T x[W];
#pragma unroll
            for (int e = 0; e < W; ++e) {
                int ls, r;
                soa_pos(vi, e, ls, r);
                x[e] = ls < ns ? tile[ls * PITCH + r] : T(0);  // pad lanes of the last block stay zero
            }
            *reinterpret_cast<VT*>(dp + vi * W) = pack(x);
        } else if (ns == 32) {
            T x[W];
#pragma unroll
            for (int e = 0; e < W; ++e) {
                int ls, r;
                aos_pos(vi, e, ls, r);
                x[e] = tile[ls * PITCH + r];
            }
            *reinterpret_cast<VT*>(dp + vi * W) = pack(x);
        } else {
#pragma unroll
            for (int e = 0; e < W; ++e) {
                int ls, r;
                aos_pos(vi, e, ls, r);
                if (ls < ns) dp[vi * W + e] = tile[ls * PITCH + r];
            }
        }
    }
}

static int transpose_launch(lqx_ctx* ctx, const lqx_field* f, const void* src, void* dst, bool to_soa) {
    return lqx_transpose_range(ctx, f->kind, f->prec, src, dst, to_soa, 0, (ctx->geo.V + 31) / 32, ctx->stream);
}

int lqx_transpose_range(lqx_ctx* ctx, lqx_kind kind, lqx_prec prec, const void* src, void* dst, bool to_soa, int blk0,
                        int nblk, cudaStream_t stream) {
    const Geo& g = ctx->geo;
    const int nreal = 2 * (int)kind;
    const int grid = (nblk + kTransposeBlocks - 1) / kTransposeBlocks, end = blk0 + nblk;
    if (grid <= 0) return LQX_OK;
#define LQX_TR(T, NREAL)                                                                                        \
    do {                                                                                                        \
        if (to_soa) k_transpose<T, NREAL, true><<<grid, 256, 0, stream>>>(g.V, blk0, end, (const T*)src, (T*)dst); \
        else k_transpose<T, NREAL, false><<<grid, 256, 0, stream>>>(g.V, blk0, end, (const T*)src, (T*)dst);       \
    } while (0)
#define LQX_TR_KIND(T)                      \
    switch (nreal) {                        \
        case 2: LQX_TR(T, 2); break;        \
        case 6: LQX_TR(T, 6); break;        \
        case 18: LQX_TR(T, 18); break;      \
        default: LQX_TR(T, 24); break;      \
    }
    if (prec == LQX_F32) { LQX_TR_KIND(float) } else { LQX_TR_KIND(double) }
#undef LQX_TR_KIND
#undef LQX_TR
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}

extern "C" int lqx_field_import_dev(lqx_field* f, const void* dev_qdp_order) {
    if (!f || !dev_qdp_order) return LQX_EINVAL;
    // the converter moves 128-bit words on both sides: a misaligned view would fault (a sticky context error)
    if (((uintptr_t)dev_qdp_order & 15) != 0) return lqx_fail(f->ctx, LQX_EINVAL, "import_dev: the device buffer must be 16-byte aligned");
    LQX_CUDA(f->ctx, cudaSetDevice(f->ctx->device));
    return transpose_launch(f->ctx, f, dev_qdp_order, f->data, true);
}
extern "C" int lqx_field_export_dev(const lqx_field* f, void* dev_qdp_order) {
    if (!f || !dev_qdp_order) return LQX_EINVAL;
    if (((uintptr_t)dev_qdp_order & 15) != 0) return lqx_fail(f->ctx, LQX_EINVAL, "export_dev: the device buffer must be 16-byte aligned");
    LQX_CUDA(f->ctx, cudaSetDevice(f->ctx->device));
    return transpose_launch(f->ctx, f, f->data, dev_qdp_order, false);
}

// staging buffer for push/pop (QDP-order copy of one field on the device): cached in the context, grow-only
static int ensure_stage(lqx_ctx* ctx, size_t bytes) {
    if (ctx->stage_cap >= bytes) return LQX_OK;
    if (ctx->stage) {
        cudaStreamSynchronize(ctx->stream);
        cudaFree(ctx->stage);
        ctx->stage = nullptr;
        ctx->stage_cap = 0;
    }
    if (cudaMalloc(&ctx->stage, bytes) != cudaSuccess) {
        cudaGetLastError();
        return lqx_fail(ctx, LQX_ENOMEM, "push/pop staging buffer");
    }
    ctx->stage_cap = bytes;
    return LQX_OK;
}

// sync = false: the copy and the conversion are only enqueued (the caller synchronises before the host buffer
// is reused or read); stream order keeps successive uses of the one staging buffer apart
int lqx_push_impl(lqx_field* f, const void* host, bool sync) {
    lqx_ctx* ctx = f->ctx;
    const size_t bytes = (size_t)ctx->geo.V * 2 * (int)f->kind * (int)f->prec;
    int rc = ensure_stage(ctx, bytes);
    if (rc) return rc;
    cudaError_t e = cudaMemcpyAsync(ctx->stage, host, bytes, cudaMemcpyHostToDevice, ctx->stream);
    if (e != cudaSuccess) return lqx_cuda_fail(ctx, e, "push H2D");
    rc = transpose_launch(ctx, f, ctx->stage, f->data, true);
    if (rc == LQX_OK && sync) {
        e = cudaStreamSynchronize(ctx->stream);  // host buffer is only touched during the call
        if (e != cudaSuccess) rc = lqx_cuda_fail(ctx, e, "push sync");
    }
    return rc;
}

int lqx_pop_impl(const lqx_field* f, void* host, bool sync) {
    lqx_ctx* ctx = f->ctx;
    const size_t bytes = (size_t)ctx->geo.V * 2 * (int)f->kind * (int)f->prec;
    int rc = ensure_stage(ctx, bytes);
    if (rc) return rc;
    rc = transpose_launch(ctx, f, f->data, ctx->stage, false);
    if (rc) return rc;
    cudaError_t e = cudaMemcpyAsync(host, ctx->stage, bytes, cudaMemcpyDeviceToHost, ctx->stream);
    if (e != cudaSuccess) return lqx_cuda_fail(ctx, e, "pop D2H");
    if (sync) {
        e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) return lqx_cuda_fail(ctx, e, "pop sync");
    }
    return LQX_OK;
}

extern "C" int lqx_field_push(lqx_field* f, const void* host) {
    if (!f || !host) return LQX_EINVAL;
    LQX_CUDA(f->ctx, cudaSetDevice(f->ctx->device));
    return lqx_push_impl(f, host, true);
}

extern "C" int lqx_field_pop(const lqx_field* f, void* host) {
    if (!f || !host) return LQX_EINVAL;
    LQX_CUDA(f->ctx, cudaSetDevice(f->ctx->device));
    return lqx_pop_impl(f, host, true);
}

// --------------------------------------------------------------------------------------------
// reduction second stage
// --------------------------------------------------------------------------------------------
int lqx_ensure_partials(lqx_ctx* ctx, size_t ndoubles) {
    if (ctx->partials_cap >= ndoubles) return LQX_OK;
    if (ctx->d_partials) {
        cudaStreamSynchronize(ctx->stream);
        cudaFree(ctx->d_partials);
        ctx->d_partials = nullptr;
        ctx->partials_cap = 0;
    }
    size_t cap = std::max<size_t>(ndoubles, 1 << 16);
    if (cudaMalloc(&ctx->d_partials, cap * sizeof(double)) != cudaSuccess) {
        cudaGetLastError();
        return lqx_fail(ctx, LQX_ENOMEM, "reduction scratch");
    }
    ctx->partials_cap = cap;
    return LQX_OK;
}

// one CTA per component; fixed strided accumulation (4 independent chains per thread) + fixed tree
__global__ void __launch_bounds__(1024) k_sum_partials(const double* __restrict__ partials, int nblocks, double* __restrict__ out) {
    __shared__ double sh[32];
    const double* p = partials + (size_t)blockIdx.x * nblocks;
    double t0 = 0.0, t1 = 0.0, t2 = 0.0, t3 = 0.0;
    int i = threadIdx.x;
    for (; i + 3 * 1024 < nblocks; i += 4 * 1024) {
        t0 += p[i];
        t1 += p[i + 1024];
        t2 += p[i + 2048];
        t3 += p[i + 3072];
    }
    for (; i < nblocks; i += 1024) t0 += p[i];
    double t = (t0 + t1) + (t2 + t3);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = t;
    __syncthreads();
    if (threadIdx.x < 32) {
        t = sh[threadIdx.x];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (threadIdx.x == 0) out[blockIdx.x] = t;
    }
}

int lqx_sum_partials(lqx_ctx* ctx, int nblocks, int ncomp, double* out) {
    k_sum_partials<<<ncomp, 1024, 0, ctx->stream>>>(ctx->d_partials, nblocks, out);
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}

int lqx_fetch_result(lqx_ctx* ctx, int n, double* out) {
    LQX_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < n; ++i) out[i] = ctx->h_result[i];
    return LQX_OK;
}
