// lqx internal declarations: context / field handles, lattice geometry with in-kernel periodic
// neighbour arithmetic, SoA addressing (a2) and the site algebra used by every
// kernel (sec.4 types; operators of Listing 1).
// Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

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
    int stride;  // plane stride in elements (V rounded up to 32)
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
    double* d_result;    // 64 doubles
    double* h_result;    // pinned, 64 doubles
    int64_t launches;
    int num_sms;
    int opt_smear_variant;
    int opt_block;
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
int lqx_cuda_fail(lqx_ctx* ctx, cudaError_t e, const char* where);
int lqx_ensure_partials(lqx_ctx* ctx, size_t ndoubles);
// second stage of every reduction: sums nblocks partials of ncomp doubles (layout
// partials[comp*nblocks + b]) into d_out[0 .. ncomp) (device memory, e.g. ctx->d_result)
int lqx_reduce_finish(lqx_ctx* ctx, int nblocks, int ncomp, double* d_out);
// copies ctx->d_result[0..n) to host `out` and synchronises the stream
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

static inline bool lqx_same(const lqx_field* a, const lqx_field* b) { return a->data == b->data; }

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
// device side: site algebra on SoA planes.  T = float or double.
// Colour matrix element (i,j): planes 2*(3*i+j) (re) and 2*(3*i+j)+1 (im).
// --------------------------------------------------------------------------------------------
template <typename T>
struct Mat3 {
    T re[3][3], im[3][3];
};
template <typename T>
struct Vec3 {
    T re[3], im[3];
};

template <typename T>
__device__ __forceinline__ Mat3<T> load_mat(const T* __restrict__ p, int stride, int s) {
    Mat3<T> m;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            m.re[i][j] = __ldg(p + (size_t)(2 * (3 * i + j)) * stride + s);
            m.im[i][j] = __ldg(p + (size_t)(2 * (3 * i + j) + 1) * stride + s);
        }
    return m;
}
template <typename T>
__device__ __forceinline__ void store_mat(T* __restrict__ p, int stride, int s, const Mat3<T>& m) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            p[(size_t)(2 * (3 * i + j)) * stride + s] = m.re[i][j];
            p[(size_t)(2 * (3 * i + j) + 1) * stride + s] = m.im[i][j];
        }
}
// vector `a` of nspin-component field: planes 2*(3*a+i)+c
template <typename T>
__device__ __forceinline__ Vec3<T> load_vec(const T* __restrict__ p, int stride, int s, int a) {
    Vec3<T> v;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        v.re[i] = __ldg(p + (size_t)(2 * (3 * a + i)) * stride + s);
        v.im[i] = __ldg(p + (size_t)(2 * (3 * a + i) + 1) * stride + s);
    }
    return v;
}
template <typename T>
__device__ __forceinline__ void store_vec(T* __restrict__ p, int stride, int s, int a, const Vec3<T>& v) {
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        p[(size_t)(2 * (3 * a + i)) * stride + s] = v.re[i];
        p[(size_t)(2 * (3 * a + i) + 1) * stride + s] = v.im[i];
    }
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
// device side: deterministic block reduction of NC doubles per thread.
// warp shuffle tree -> shared memory across warps -> thread 0 writes partials[c*nblocks + block].
// --------------------------------------------------------------------------------------------
template <int NC>
__device__ __forceinline__ void block_reduce_store(double (&v)[NC], double* __restrict__ partials,
                                                   int nblocks, int block) {
    __shared__ double sh[32][NC + (NC % 2 == 0 ? 1 : 0)];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nwarps = (blockDim.x + 31) >> 5;
    __syncthreads();  // the buffer may be reused by a second call in the same kernel
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
