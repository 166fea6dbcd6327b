// lqx internal declarations: context / field handles, lattice geometry with in-kernel periodic
// neighbour arithmetic, blocked-SoA addressing (a2) and the site algebra used by every
// kernel (sec.4 types; operators of Listing 1).
// Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <string>
#include <utility>
#include <vector>

#include "../../include/lqx.h"

// --------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------
struct FastDiv {  // floor(n/d) for 0 <= n < 2^31 as (n*mul) >> (31+sh); mul = ceil(2^(31+sh)/d)
    uint32_t mul;
    uint32_t sh;
    uint32_t d;
};

struct Geo {  // passed by value to kernels
    int L[4];
    int stride_site[4];  // 1, L0, L0*L1, L0*L1*L2
    int V;
    int Vpad;    // V rounded up to a whole number of 32-site blocks
    FastDiv d0, d1, d2;
};

struct lqx_ctx {
    Geo geo;
    int device;
    cudaStream_t stream;
    std::string last_error;
    std::vector<lqx_field*> fields;
    double* d_partials;  // reduction scratch
    size_t partials_cap; // in doubles
    double* d_result;    // 64 doubles (device scratch results)
    double* h_result;    // pinned + mapped, 64 doubles: kernels write results straight to the host
    lqx_field* host_work[12];  // work fields of lqx_smear_iterate_host, kept between calls: links, ping-pong
                               // scratch, and (streamed one-step path) four QDP-order staging fields
    cudaStream_t pipe_stream[2];          // upload and download streams of the streamed host path (lazy)
    std::vector<cudaEvent_t> pipe_events; // its per-slab events (lazy, no timing)
    int opt_host_slabs;                   // -1 = automatic, 0 = off (serial push / step / pop), n = at most n slabs
    void* stage;       // device staging buffer of push/pop (one field in QDP order), grow-only
    size_t stage_cap;
    unsigned int* d_ticket;  // last-block ticket of the one-launch reductions (zero between launches)
    int64_t launches;
    int num_sms;
    int opt_smear_variant;
    int opt_plaq_variant;                 // plaquette kernel: 0 = automatic, 1 = rolled loops, 2 = the site's four links held in registers
    int opt_block;
    int opt_hop_block;                    // CTA size of the hop kernel on linear blocks: 0 = default (128), 32, 64, 128, 256
    int opt_jacobi_block, opt_jacobi_sites;  // launch geometry of the Jacobi step (0 = default 128 x 1)
    int opt_tile;  // -1 = automatic, 0 = Linear, 1..3 = TileA..TileC (lqx_smear.cuh)
    int opt_bulk_fill;  // row-tile smear kernel: 1 = fill the tile by TMA bulk copies where its rows are whole blocks (measured slower), 0 = cp.async
    // launch geometries kept by lqx_autotune (lqx_tune.cu), per precision (0 = fp32, 1 = fp64); 0 / -1 = not tuned.
    // An explicit option always wins over a tuned value, a tuned value over the built-in default.
    int tuned_smear_variant[2], tuned_smear_tile[2];
    int tuned_plaq_variant[2];
    int tuned_hop_block[2];
    int tuned_jacobi_block[2], tuned_jacobi_sites[2];
    // what the last smear launch ran (bench.py reports the kernel and its executed lane-ops from here)
    int last_smear_variant, last_smear_lane_ops;
    const char* last_smear_kernel;
    // optional per-kernel-class device timing (bench harness): cudaEvent pairs on the stream
    bool timing;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> timers[LQX_NUM_KERNEL_CLASSES];
};

// RAII: brackets the kernel launches of one class with events when ctx->timing is on
struct LqxTimed {
    lqx_ctx* ctx;
    cudaEvent_t stop;
    LqxTimed(lqx_ctx* c, int which) : ctx(c), stop(nullptr) {
        if (!c->timing) return;
        cudaEvent_t start;
        if (cudaEventCreate(&start) != cudaSuccess || cudaEventCreate(&stop) != cudaSuccess) {
            stop = nullptr;
            return;
        }
        cudaEventRecord(start, c->stream);
        c->timers[which].push_back(std::make_pair(start, stop));
    }
    ~LqxTimed() {
        if (stop) cudaEventRecord(stop, ctx->stream);
    }
};

struct lqx_field {
    lqx_ctx* ctx;
    lqx_kind kind;
    lqx_prec prec;
    void* data;
    bool owned;
};

int lqx_fail(lqx_ctx* ctx, int code, const char* what);
int lqx_push_impl(lqx_field* f, const void* host, bool sync);  // lqx_core.cu; sync = false only enqueues
int lqx_pop_impl(const lqx_field* f, void* host, bool sync);
// QDP order <-> blocked layout for the 32-site blocks [blk0, blk0 + nblk) of a field, on `stream` (lqx_core.cu)
int lqx_transpose_range(lqx_ctx* ctx, lqx_kind kind, lqx_prec prec, const void* src, void* dst, bool to_soa, int blk0,
                        int nblk, cudaStream_t stream);
void lqx_jit_release(lqx_ctx* ctx);
void lqx_staged_release(lqx_ctx* ctx);  // frees the staged smear kernel's tables (lqx_smear_staged.cu)  // unloads the context's run-time compiled expression kernels (lqx_jit.cu)
int lqx_cuda_fail(lqx_ctx* ctx, cudaError_t e, const char* where);
int lqx_ensure_partials(lqx_ctx* ctx, size_t ndoubles);
// synchronises the stream and copies ctx->h_result[0..n) (written by a reduction kernel) to `out`
int lqx_fetch_result(lqx_ctx* ctx, int n, double* out);

#define LQX_CUDA(ctx, call)                                              \
    do {                                                                 \
        cudaError_t e__ = (call);                                        \
        if (e__ != cudaSuccess) return lqx_cuda_fail((ctx), e__, #call); \
    } while (0)

#define LQX_LAUNCH_CHECK(ctx)                                                  \
    do {                                                                       \
        (ctx)->launches++;                                                     \
        cudaError_t e__ = cudaGetLastError();                                  \
        if (e__ != cudaSuccess) return lqx_cuda_fail((ctx), e__, "kernel launch"); \
    } while (0)

// Aliasing between two fields is decided on BYTE RANGES (two lqx_field_attach views may overlap without sharing
// a base pointer).  lqx_same: any overlap -- what the shifted forms reject with LQX_EALIAS.  lqx_identical: the same
// storage exactly -- the only aliasing a site-local form may run with (in place, reading A21); those launches use
// the plain-load, non-__restrict__ instantiation of their kernel (ld.global.nc is defined only for memory the
// kernel never writes).
static inline size_t lqx_field_nbytes(const lqx_field* f) {
    return (size_t)f->ctx->geo.Vpad * 2 * (size_t)(int)f->kind * (size_t)(int)f->prec;
}
static inline bool lqx_same(const lqx_field* a, const lqx_field* b) {
    const char* pa = (const char*)a->data;
    const char* pb = (const char*)b->data;
    return pa < pb + lqx_field_nbytes(b) && pb < pa + lqx_field_nbytes(a);
}
static inline bool lqx_identical(const lqx_field* a, const lqx_field* b) {
    return a->data == b->data && lqx_field_nbytes(a) == lqx_field_nbytes(b);
}
// kernel parameter types: read-only / restrict for out-of-place launches, plain for in-place ones
template <typename T, bool INPLACE>
struct KPtr {
    typedef const T* __restrict__ in;
    typedef T* __restrict__ out;
};
template <typename T>
struct KPtr<T, true> {
    typedef const T* in;
    typedef T* out;
};

// --------------------------------------------------------------------------------------------
// device side: geometry
// --------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t fdiv(uint32_t n, const FastDiv& f) {
    return (uint32_t)(((uint64_t)n * f.mul) >> (31 + f.sh));
}

// x(s): site(x) = x0 + L0*(x1 + L1*(x2 + L2*x3))
__device__ __forceinline__ void site_coords(const Geo& g, int s, int x[4]) {
    uint32_t q0 = fdiv((uint32_t)s, g.d0);
    x[0] = s - (int)q0 * g.L[0];
    uint32_t q1 = fdiv(q0, g.d1);
    x[1] = (int)q0 - (int)q1 * g.L[1];
    uint32_t q2 = fdiv(q1, g.d2);
    x[2] = (int)q1 - (int)q2 * g.L[2];
    x[3] = (int)q2;
}
// site index of x + mu^ / x - mu^ (periodic).  x[] is read through selects so that a run-time mu
// does not force the coordinates into local memory.
__device__ __forceinline__ int coord_of(const int x[4], int mu) {
    return mu == 0 ? x[0] : (mu == 1 ? x[1] : (mu == 2 ? x[2] : x[3]));
}
__device__ __forceinline__ int nbr_fwd(const Geo& g, int s, const int x[4], int mu) {
    return (coord_of(x, mu) + 1 == g.L[mu]) ? s - (g.L[mu] - 1) * g.stride_site[mu] : s + g.stride_site[mu];
}
__device__ __forceinline__ int nbr_bwd(const Geo& g, int s, const int x[4], int mu) {
    return (coord_of(x, mu) == 0) ? s + (g.L[mu] - 1) * g.stride_site[mu] : s - g.stride_site[mu];
}

// --------------------------------------------------------------------------------------------
// device side: the field store's internal layout -- blocked site-fastest SoA.
//
// Sites are grouped in blocks of 32 consecutive lexicographic sites (one warp).  Inside a block
// the NREAL reals of a site object (QDP order, lqx.h) are cut into 128-bit chunks of
// W = 16/sizeof(T) reals (4 floats / 2 doubles); chunk q of all 32 sites is contiguous:
//
//     offset(site s, real r) = (s>>5)*32*NREAL + q*32*W + (s&31)*w_q + (r - q*W),   q = r / W,
//     w_q = W for the NREAL/W full chunks, and 2 for the trailing half chunk (fp32, NREAL%4 == 2).
//
// So a warp reading one chunk of 32 consecutive sites issues ONE 128-bit load per lane over 512
// contiguous bytes, a whole colour matrix is 5 (fp32) / 9 (fp64) loads from ONE computed address
// plus immediates, and a field is exactly as large as in plain SoA (Vpad*NREAL reals).
// --------------------------------------------------------------------------------------------
template <typename T>
struct Vec128;
template <>
struct Vec128<float> {
    typedef float4 type;
    static constexpr int W = 4;
};
template <>
struct Vec128<double> {
    typedef double2 type;
    static constexpr int W = 2;
};

__device__ __forceinline__ void unpack(const float4& v, float* r) { r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w; }
__device__ __forceinline__ void unpack(const double2& v, double* r) { r[0] = v.x; r[1] = v.y; }
__device__ __forceinline__ float4 pack(const float* r) { return make_float4(r[0], r[1], r[2], r[3]); }
__device__ __forceinline__ double2 pack(const double* r) { return make_double2(r[0], r[1]); }

// element offset of (site s, real r) for a field of nreal reals per site, W reals per 128 bits
__host__ __device__ __forceinline__ size_t lqx_layout_offset(int s, int r, int nreal, int W) {
    const int nfull = nreal / W;
    const int q = r / W < nfull ? r / W : nfull;
    const int wq = q < nfull ? W : nreal - nfull * W;
    return (size_t)(s >> 5) * 32 * nreal + (size_t)q * 32 * W + (size_t)(s & 31) * wq + (r - q * W);
}

// 128-bit / 64-bit read-only loads as VOLATILE asm: the compiler keeps them in program order, which
// is how the unrolled nearest-neighbour kernels control how many operands are in flight.
__device__ __forceinline__ float4 ldg_pinned(const float4* p) {
    float4 v;
    asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ double2 ldg_pinned(const double2* p) {
    double2 v;
    asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ float2 ldg_pinned(const float2* p) {
    float2 v;
    asm volatile("ld.global.nc.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}

// all NREAL reals of site s: through the read-only path (ld.global.nc), or with plain loads (PLAIN) where the same
// kernel writes the field (in-place site-local forms)
template <typename T, int NREAL, bool PLAIN = false>
__device__ __forceinline__ void load_site(const T* base, int s, T (&r)[NREAL]) {
    typedef typename Vec128<T>::type V;
    constexpr int W = Vec128<T>::W, NFULL = NREAL / W;
    const T* blk = base + (size_t)(s >> 5) * (32 * NREAL);
    const int lane = s & 31;
    const V* p = reinterpret_cast<const V*>(blk) + lane;
#pragma unroll
    for (int q = 0; q < NFULL; ++q) unpack(PLAIN ? p[q * 32] : __ldg(p + q * 32), &r[q * W]);
    if (NREAL % W != 0) {  // fp32 only: trailing (re,im) pair
        const float2* ph = reinterpret_cast<const float2*>(blk + NFULL * 32 * W) + lane;
        const float2 t = PLAIN ? *ph : __ldg(ph);
        r[NFULL * W] = (T)t.x;
        r[NFULL * W + 1] = (T)t.y;
    }
}
template <typename T, int NREAL>
__device__ __forceinline__ void load_site_pinned(const T* __restrict__ base, int s, T (&r)[NREAL]) {
    typedef typename Vec128<T>::type V;
    constexpr int W = Vec128<T>::W, NFULL = NREAL / W;
    const T* blk = base + (size_t)(s >> 5) * (32 * NREAL);
    const int lane = s & 31;
    const V* p = reinterpret_cast<const V*>(blk) + lane;
#pragma unroll
    for (int q = 0; q < NFULL; ++q) unpack(ldg_pinned(p + q * 32), &r[q * W]);
    if (NREAL % W != 0) {
        const float2 t = ldg_pinned(reinterpret_cast<const float2*>(blk + NFULL * 32 * W) + lane);
        r[NFULL * W] = (T)t.x;
        r[NFULL * W + 1] = (T)t.y;
    }
}
// STREAM: st.global.cs (evict-first) for results that no later part of the same pass reads
template <typename T, int NREAL, bool STREAM = false>
__device__ __forceinline__ void store_site(T* base, int s, const T (&r)[NREAL]) {
    typedef typename Vec128<T>::type V;
    constexpr int W = Vec128<T>::W, NFULL = NREAL / W;
    T* blk = base + (size_t)(s >> 5) * (32 * NREAL);
    const int lane = s & 31;
    V* p = reinterpret_cast<V*>(blk) + lane;
#pragma unroll
    for (int q = 0; q < NFULL; ++q) {
        if (STREAM) __stcs(p + q * 32, pack(&r[q * W]));
        else p[q * 32] = pack(&r[q * W]);
    }
    if (NREAL % W != 0) {
        const float2 h = make_float2((float)r[NFULL * W], (float)r[NFULL * W + 1]);
        if (STREAM) __stcs(reinterpret_cast<float2*>(blk + NFULL * 32 * W) + lane, h);
        else reinterpret_cast<float2*>(blk + NFULL * 32 * W)[lane] = h;
    }
}

// reals [R0, R0+NR) of site s of a field with NREAL reals per site (whole 128-bit chunks only)
template <typename T, int NREAL, int R0, int NR>
__device__ __forceinline__ void load_site_part(const T* __restrict__ base, int s, T (&r)[NR]) {
    typedef typename Vec128<T>::type V;
    constexpr int W = Vec128<T>::W;
    static_assert(R0 % W == 0 && NR % W == 0 && R0 + NR <= (NREAL / W) * W, "whole chunks only");
    const V* p = reinterpret_cast<const V*>(base + (size_t)(s >> 5) * (32 * NREAL)) + (s & 31);
#pragma unroll
    for (int q = 0; q < NR / W; ++q) unpack(__ldg(p + (R0 / W + q) * 32), &r[q * W]);
}
template <typename T, int NREAL, int R0, int NR>
__device__ __forceinline__ void store_site_part(T* __restrict__ base, int s, const T (&r)[NR]) {
    typedef typename Vec128<T>::type V;
    constexpr int W = Vec128<T>::W;
    static_assert(R0 % W == 0 && NR % W == 0 && R0 + NR <= (NREAL / W) * W, "whole chunks only");
    V* p = reinterpret_cast<V*>(base + (size_t)(s >> 5) * (32 * NREAL)) + (s & 31);
#pragma unroll
    for (int q = 0; q < NR / W; ++q) p[(R0 / W + q) * 32] = pack(&r[q * W]);
}

// --------------------------------------------------------------------------------------------
// device side: site algebra.  T = float or double.
// Colour matrix element (i,j): QDP-order reals 2*(3*i+j) (re) and 2*(3*i+j)+1 (im).
// --------------------------------------------------------------------------------------------
template <typename T>
struct Mat3 {
    T re[3][3], im[3][3];
};
template <typename T>
struct Vec3 {
    T re[3], im[3];
};

template <typename T, bool PLAIN = false>
__device__ __forceinline__ Mat3<T> load_mat(const T* p, int s) {
    T r[18];
    load_site<T, 18, PLAIN>(p, s, r);
    Mat3<T> m;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            m.re[i][j] = r[2 * (3 * i + j)];
            m.im[i][j] = r[2 * (3 * i + j) + 1];
        }
    return m;
}
template <typename T>
__device__ __forceinline__ Mat3<T> load_mat_pinned(const T* __restrict__ p, int s) {
    T r[18];
    load_site_pinned<T, 18>(p, s, r);
    Mat3<T> m;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            m.re[i][j] = r[2 * (3 * i + j)];
            m.im[i][j] = r[2 * (3 * i + j) + 1];
        }
    return m;
}
template <typename T>
__device__ __forceinline__ void store_mat(T* p, int s, const Mat3<T>& m) {
    T r[18];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            r[2 * (3 * i + j)] = m.re[i][j];
            r[2 * (3 * i + j) + 1] = m.im[i][j];
        }
    store_site<T, 18>(p, s, r);
}
// NSPIN colour vectors of one site (NSPIN = 1: LatticeColorVector, 4: LatticeFermion)
template <typename T, int NSPIN, bool PLAIN = false>
__device__ __forceinline__ void load_vecs(const T* p, int s, Vec3<T> (&v)[NSPIN]) {
    T r[6 * NSPIN];
    load_site<T, 6 * NSPIN, PLAIN>(p, s, r);
#pragma unroll
    for (int a = 0; a < NSPIN; ++a)
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            v[a].re[i] = r[2 * (3 * a + i)];
            v[a].im[i] = r[2 * (3 * a + i) + 1];
        }
}
template <typename T, int NSPIN, bool STREAM = false>
__device__ __forceinline__ void store_vecs(T* p, int s, const Vec3<T> (&v)[NSPIN]) {
    T r[6 * NSPIN];
#pragma unroll
    for (int a = 0; a < NSPIN; ++a)
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            r[2 * (3 * a + i)] = v[a].re[i];
            r[2 * (3 * a + i) + 1] = v[a].im[i];
        }
    store_site<T, 6 * NSPIN, STREAM>(p, s, r);
}

// C = A*B        (AB)_ij = sum_k A_ik B_kj
template <typename T>
__device__ __forceinline__ Mat3<T> mul_nn(const Mat3<T>& a, const Mat3<T>& b) {
    Mat3<T> c;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            T re = a.re[i][0] * b.re[0][j];
            T im = a.re[i][0] * b.im[0][j];
            re = fma(-a.im[i][0], b.im[0][j], re);
            im = fma(a.im[i][0], b.re[0][j], im);
#pragma unroll
            for (int k = 1; k < 3; ++k) {
                re = fma(a.re[i][k], b.re[k][j], re);
                im = fma(a.re[i][k], b.im[k][j], im);
                re = fma(-a.im[i][k], b.im[k][j], re);
                im = fma(a.im[i][k], b.re[k][j], im);
            }
            c.re[i][j] = re;
            c.im[i][j] = im;
        }
    return c;
}
// C += A*B
template <typename T>
__device__ __forceinline__ void mac_nn(Mat3<T>& c, const Mat3<T>& a, const Mat3<T>& b) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            T re = c.re[i][j], im = c.im[i][j];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                re = fma(a.re[i][k], b.re[k][j], re);
                im = fma(a.re[i][k], b.im[k][j], im);
                re = fma(-a.im[i][k], b.im[k][j], re);
                im = fma(a.im[i][k], b.re[k][j], im);
            }
            c.re[i][j] = re;
            c.im[i][j] = im;
        }
}
// C += A*adj(B)   (A B^dag)_ij = sum_k A_ik conj(B_jk)
template <typename T>
__device__ __forceinline__ void mac_na(Mat3<T>& c, const Mat3<T>& a, const Mat3<T>& b) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            T re = c.re[i][j], im = c.im[i][j];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                re = fma(a.re[i][k], b.re[j][k], re);
                im = fma(a.im[i][k], b.re[j][k], im);
                re = fma(a.im[i][k], b.im[j][k], re);
                im = fma(-a.re[i][k], b.im[j][k], im);
            }
            c.re[i][j] = re;
            c.im[i][j] = im;
        }
}
// C += adj(A)*B   (A^dag B)_ij = sum_k conj(A_ki) B_kj
template <typename T>
__device__ __forceinline__ void mac_an(Mat3<T>& c, const Mat3<T>& a, const Mat3<T>& b) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            T re = c.re[i][j], im = c.im[i][j];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                re = fma(a.re[k][i], b.re[k][j], re);
                im = fma(a.re[k][i], b.im[k][j], im);
                re = fma(a.im[k][i], b.im[k][j], re);
                im = fma(-a.im[k][i], b.re[k][j], im);
            }
            c.re[i][j] = re;
            c.im[i][j] = im;
        }
}
// --------------------------------------------------------------------------------------------
// fp32: the same products on packed (re, im) pairs.  sm_100a has FFMA2 (PTX fma.rn.f32x2): two fp32
// FMAs per issue slot on a 64-bit register pair, and its SASS operand forms cover a complex
// multiply-accumulate without any data movement: a 32-bit register broadcast to both lanes (.F32),
// the pair swapped (.LO_HI) and a per-lane sign (.NP / .PN) -- ptxas folds mov.b64 {x, x},
// {y, x} and {-y, x} into them as long as the signed pair is the FIRST multiplicand.  So
//     c += a*b :  c = fma2((b.re, b.im), a.re, c);  c = fma2((-b.im, b.re), a.im, c)
// is two instructions instead of four, with the operands exactly as the 128-bit loads deliver them.
// Same lane throughput as scalar FFMA, half the issue slots (profiles/r02a).  Every lane is an IEEE
// fma in the order of the generic code above except that in mac_na the two im terms swap.
// --------------------------------------------------------------------------------------------
typedef unsigned long long f32x2_t;
__device__ __forceinline__ f32x2_t pk2(float lo, float hi) {
    f32x2_t d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ void upk2(f32x2_t d, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(d)); }
__device__ __forceinline__ f32x2_t fma2(f32x2_t a, f32x2_t b, f32x2_t c) {
    f32x2_t d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2_t mul2(f32x2_t a, f32x2_t b) {
    f32x2_t d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
// c += a*b, c += a*conj(b), c += conj(a)*b on c = (re, im)
__device__ __forceinline__ f32x2_t cmac_nn(f32x2_t c, float ar, float ai, float br, float bi) {
    c = fma2(pk2(br, bi), pk2(ar, ar), c);
    return fma2(pk2(-bi, br), pk2(ai, ai), c);
}
__device__ __forceinline__ f32x2_t cmac_nc(f32x2_t c, float ar, float ai, float br, float bi) {
    c = fma2(pk2(br, -bi), pk2(ar, ar), c);
    return fma2(pk2(bi, br), pk2(ai, ai), c);
}
__device__ __forceinline__ f32x2_t cmac_cn(f32x2_t c, float ar, float ai, float br, float bi) {
    c = fma2(pk2(br, bi), pk2(ar, ar), c);
    return fma2(pk2(bi, -br), pk2(ai, ai), c);
}
// non-template overloads: chosen over the templates above for T = float
__device__ __forceinline__ Mat3<float> mul_nn(const Mat3<float>& a, const Mat3<float>& b) {
    Mat3<float> c;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            f32x2_t t = mul2(pk2(b.re[0][j], b.im[0][j]), pk2(a.re[i][0], a.re[i][0]));
            t = fma2(pk2(-b.im[0][j], b.re[0][j]), pk2(a.im[i][0], a.im[i][0]), t);
#pragma unroll
            for (int k = 1; k < 3; ++k) t = cmac_nn(t, a.re[i][k], a.im[i][k], b.re[k][j], b.im[k][j]);
            upk2(t, c.re[i][j], c.im[i][j]);
        }
    return c;
}
__device__ __forceinline__ void mac_nn(Mat3<float>& c, const Mat3<float>& a, const Mat3<float>& b) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            f32x2_t t = pk2(c.re[i][j], c.im[i][j]);
#pragma unroll
            for (int k = 0; k < 3; ++k) t = cmac_nn(t, a.re[i][k], a.im[i][k], b.re[k][j], b.im[k][j]);
            upk2(t, c.re[i][j], c.im[i][j]);
        }
}
__device__ __forceinline__ void mac_na(Mat3<float>& c, const Mat3<float>& a, const Mat3<float>& b) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            f32x2_t t = pk2(c.re[i][j], c.im[i][j]);
#pragma unroll
            for (int k = 0; k < 3; ++k) t = cmac_nc(t, a.re[i][k], a.im[i][k], b.re[j][k], b.im[j][k]);
            upk2(t, c.re[i][j], c.im[i][j]);
        }
}
__device__ __forceinline__ void mac_an(Mat3<float>& c, const Mat3<float>& a, const Mat3<float>& b) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            f32x2_t t = pk2(c.re[i][j], c.im[i][j]);
#pragma unroll
            for (int k = 0; k < 3; ++k) t = cmac_cn(t, a.re[k][i], a.im[k][i], b.re[k][j], b.im[k][j]);
            upk2(t, c.re[i][j], c.im[i][j]);
        }
}
__device__ __forceinline__ void mac_mv(Vec3<float>& w, const Mat3<float>& m, const Vec3<float>& v) {
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        f32x2_t t = pk2(w.re[i], w.im[i]);
#pragma unroll
        for (int j = 0; j < 3; ++j) t = cmac_nn(t, m.re[i][j], m.im[i][j], v.re[j], v.im[j]);
        upk2(t, w.re[i], w.im[i]);
    }
}
__device__ __forceinline__ void mac_adj_mv(Vec3<float>& w, const Mat3<float>& m, const Vec3<float>& v) {
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        f32x2_t t = pk2(w.re[i], w.im[i]);
#pragma unroll
        for (int j = 0; j < 3; ++j) t = cmac_cn(t, m.re[j][i], m.im[j][i], v.re[j], v.im[j]);
        upk2(t, w.re[i], w.im[i]);
    }
}

template <typename T>
__device__ __forceinline__ Mat3<T> zero_mat() {
    Mat3<T> c;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            c.re[i][j] = T(0);
            c.im[i][j] = T(0);
        }
    return c;
}
template <typename T>
__device__ __forceinline__ Mat3<T> mul_na(const Mat3<T>& a, const Mat3<T>& b) {
    Mat3<T> c = zero_mat<T>();
    mac_na(c, a, b);
    return c;
}
template <typename T>
__device__ __forceinline__ Mat3<T> mul_an(const Mat3<T>& a, const Mat3<T>& b) {
    Mat3<T> c = zero_mat<T>();
    mac_an(c, a, b);
    return c;
}
// Re tr(A * adj(B)) = sum_ij Re(A_ij conj(B_ij))
template <typename T>
__device__ __forceinline__ T re_tr_na(const Mat3<T>& a, const Mat3<T>& b) {
    T t = T(0);
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            t = fma(a.re[i][j], b.re[i][j], t);
            t = fma(a.im[i][j], b.im[i][j], t);
        }
    return t;
}
// w += M v  /  w += adj(M) v
template <typename T>
__device__ __forceinline__ void mac_mv(Vec3<T>& w, const Mat3<T>& m, const Vec3<T>& v) {
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        T re = w.re[i], im = w.im[i];
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            re = fma(m.re[i][j], v.re[j], re);
            im = fma(m.re[i][j], v.im[j], im);
            re = fma(-m.im[i][j], v.im[j], re);
            im = fma(m.im[i][j], v.re[j], im);
        }
        w.re[i] = re;
        w.im[i] = im;
    }
}
template <typename T>
__device__ __forceinline__ void mac_adj_mv(Vec3<T>& w, const Mat3<T>& m, const Vec3<T>& v) {
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        T re = w.re[i], im = w.im[i];
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            re = fma(m.re[j][i], v.re[j], re);
            im = fma(m.re[j][i], v.im[j], im);
            re = fma(m.im[j][i], v.im[j], re);
            im = fma(-m.im[j][i], v.re[j], im);
        }
        w.re[i] = re;
        w.im[i] = im;
    }
}

// --------------------------------------------------------------------------------------------
// device side: deterministic reduction of NC doubles per thread in ONE launch.
// warp shuffle tree -> shared memory across warps -> partials[c*nblocks + block]; the block that
// takes the last ticket sums the partials in a fixed order and writes out[0..NC).  The grid is a
// fixed function of the lattice, so the summation tree (and the result) is the same run to run.
// `out` may be device memory or pinned host memory (UVA).
// --------------------------------------------------------------------------------------------
template <int NC>
__device__ __forceinline__ void block_reduce_finish(double (&v)[NC], double* __restrict__ partials,
                                                    unsigned int* __restrict__ ticket, double* __restrict__ out) {
    __shared__ double sh[32][NC + (NC % 2 == 0 ? 1 : 0)];
    __shared__ bool last;
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int nthreads = blockDim.x * blockDim.y * blockDim.z;
    const int lane = tid & 31, warp = tid >> 5;
    const int nwarps = (nthreads + 31) >> 5;
    const int nblocks = gridDim.x * gridDim.y * gridDim.z;
    const int block = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z);
    __syncthreads();
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        double t = v[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (lane == 0) sh[warp][c] = t;
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            double t = (lane < nwarps) ? sh[lane][c] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
            if (lane == 0) partials[(size_t)c * nblocks + block] = t;
        }
        if (lane == 0) {
            // release-only ticket: orders this lane's partial stores before the increment without the
            // L1 invalidation (CCTL.IVALL) that __threadfence() would cost every CTA of the grid --
            // in the smear kernel that wipes the neighbours its co-resident CTAs share
            unsigned int t;
            asm volatile("atom.release.gpu.global.add.u32 %0, [%1], 1;" : "=r"(t) : "l"(ticket) : "memory");
            last = (t == (unsigned)(nblocks - 1));
        }
    }
    __syncthreads();
    if (!last) return;
    __threadfence();  // acquire side, paid by the one finishing CTA; partials are then read from L2
    if (NC <= 2) {  // few components: the whole CTA sums each one
        for (int c = 0; c < NC; ++c) {
            double t = 0.0;
            for (int i = tid; i < nblocks; i += nthreads) t += __ldcg(partials + (size_t)c * nblocks + i);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
            __syncthreads();
            if (lane == 0) sh[warp][0] = t;
            __syncthreads();
            if (warp == 0) {
                t = (lane < nwarps) ? sh[lane][0] : 0.0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
                if (lane == 0) out[c] = t;
            }
        }
    } else {  // many components (sum of a site object): one warp per component, all in parallel
        for (int c = warp; c < NC; c += nwarps) {
            const double* pc = partials + (size_t)c * nblocks;
            double t0 = 0.0, t1 = 0.0, t2 = 0.0, t3 = 0.0;
            int i = lane;
            for (; i + 96 < nblocks; i += 128) {
                t0 += __ldcg(pc + i);
                t1 += __ldcg(pc + i + 32);
                t2 += __ldcg(pc + i + 64);
                t3 += __ldcg(pc + i + 96);
            }
            for (; i < nblocks; i += 32) t0 += __ldcg(pc + i);
            double t = (t0 + t1) + (t2 + t3);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
            if (lane == 0) out[c] = t;
        }
        __syncthreads();
    }
    if (tid == 0) *ticket = 0u;  // ready for the next launch on this stream
}

// Two-launch form for the long nearest-neighbour kernels: the CTA only stores its partial (no fence,
// no ticket, nothing that delays its retirement); lqx_sum_partials() then adds them up in a fixed
// order with one small CTA per component.
template <int NC>
__device__ __forceinline__ void block_reduce_partial(double (&v)[NC], double* __restrict__ partials) {
    __shared__ double sh[32][NC + (NC % 2 == 0 ? 1 : 0)];
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int nthreads = blockDim.x * blockDim.y * blockDim.z;
    const int lane = tid & 31, warp = tid >> 5;
    const int nwarps = (nthreads + 31) >> 5;
    const int nblocks = gridDim.x * gridDim.y * gridDim.z;
    const int block = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z);
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        double t = v[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (lane == 0) sh[warp][c] = t;
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            double t = (lane < nwarps) ? sh[lane][c] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
            if (lane == 0) partials[(size_t)c * nblocks + block] = t;
        }
    }
}
// out[c] = sum_b partials[c*nblocks + b], c < ncomp, on the context's stream (lqx_core.cu)
int lqx_sum_partials(lqx_ctx* ctx, int nblocks, int ncomp, double* out);

// --------------------------------------------------------------------------------------------
// device side: CTA -> sites maps of the nearest-neighbour kernels (hop, plaquette, smear).
//
// Tiled<TX,TY,TZ,TT>: a CTA owns a compact 4-d tile (one thread per site, x fastest inside the
//   tile) so that the neighbour operands its threads share are served by L1.  Tiles are visited
//   x, y, z fastest inside a slab of `zs` z-tiles, then t, then the next slab: the +-t neighbour
//   slices of a slab (a few MB) are still in L2 when they are needed again, and only the two
//   z-faces of a slab are re-read from HBM.
// Linear: generic fallback for extents no tile shape divides: 128 consecutive lexicographic sites.
// --------------------------------------------------------------------------------------------
struct TileMap {
    int nt[4];   // tiles per direction (nt[3]: t-tiles this launch covers)
    int zs;      // z-tiles per slab
    int toff;    // first t-tile of the launch (a launch may cover a range of time slices, see restrict_t)
    int s0, s1;  // Linear: site range of the launch
};

template <int TX, int TY, int TZ, int TT>
struct Tiled {
    static constexpr int THREADS = TX * TY * TZ * TT;
    static constexpr int T0 = TX, T1 = TY, T2 = TZ, T3 = TT;
    __device__ static __forceinline__ bool site(const Geo& g, const TileMap& m, int x[4], int& s) {
        const int id = blockIdx.x;
        const int n01 = m.nt[0] * m.nt[1];
        const int per_slab = n01 * m.zs * m.nt[3];
        const int k = id / per_slab;
        int rem = id - k * per_slab;
        const int zsk = min(m.zs, m.nt[2] - k * m.zs);
        const int slice = n01 * zsk;
        const int tt = rem / slice;
        rem -= tt * slice;
        const int tz = rem / n01;
        rem -= tz * n01;
        const int ty = rem / m.nt[0];
        const int tx = rem - ty * m.nt[0];
        const int l = threadIdx.x;
        x[0] = tx * TX + (l % TX);
        x[1] = ty * TY + (l / TX) % TY;
        x[2] = (tz + k * m.zs) * TZ + (l / (TX * TY)) % TZ;
        x[3] = (tt + m.toff) * TT + l / (TX * TY * TZ);
        s = x[0] + g.L[0] * (x[1] + g.L[1] * (x[2] + g.L[2] * x[3]));
        return true;
    }
    static bool fits(const Geo& g) { return g.L[0] % TX == 0 && g.L[1] % TY == 0 && g.L[2] % TZ == 0 && g.L[3] % TT == 0; }
    static int grid(const Geo& g) { return (g.L[0] / TX) * (g.L[1] / TY) * (g.L[2] / TZ) * (g.L[3] / TT); }
    // restrict the launch to the time slices [t0, t1) (both multiples of TT); returns its grid size
    static int restrict_t(const Geo&, TileMap& m, int t0, int t1) {
        m.toff = t0 / TT;
        m.nt[3] = (t1 - t0) / TT;
        return m.nt[0] * m.nt[1] * m.nt[2] * m.nt[3];
    }
    static bool splits_t(int t) { return t % TT == 0; }
    static TileMap map(const Geo& g, int slab_sites_z) {
        TileMap m;
        m.nt[0] = g.L[0] / TX;
        m.nt[1] = g.L[1] / TY;
        m.nt[2] = g.L[2] / TZ;
        m.nt[3] = g.L[3] / TT;
        m.zs = std::max(1, std::min(m.nt[2], slab_sites_z / TZ));
        m.toff = 0;
        m.s0 = 0;
        m.s1 = g.V;
        return m;
    }
};

template <int NTHREADS>
struct LinearN {
    static constexpr int THREADS = NTHREADS;
    __device__ static __forceinline__ bool site(const Geo& g, const TileMap& m, int x[4], int& s) {
        s = m.s0 + blockIdx.x * THREADS + threadIdx.x;
        if (s >= m.s1) return false;
        site_coords(g, s, x);
        return true;
    }
    static bool fits(const Geo&) { return true; }
    static int grid(const Geo& g) { return (g.V + THREADS - 1) / THREADS; }
    static TileMap map(const Geo& g, int) {
        TileMap m = {{0, 0, 0, 0}, 1, 0, 0, g.V};
        return m;
    }
    static int restrict_t(const Geo& g, TileMap& m, int t0, int t1) {
        const int v3 = g.L[0] * g.L[1] * g.L[2];
        m.s0 = t0 * v3;
        m.s1 = t1 * v3;
        return (m.s1 - m.s0 + THREADS - 1) / THREADS;
    }
    static bool splits_t(int) { return true; }
};
typedef LinearN<128> Linear;
