// lqx run-time expression fusion -- the paper's own mechanism rebuilt for sm_100a:
// an expression over lattice-wide objects arrives as a flattened POD tree, the
// library generates ONE fused CUDA kernel for it (the whole expression per site, no temporaries,
// PAPER.md:61-63, :115; shifts read their operand at the periodic neighbour), compiles it at
// run time ("code generator -> NVCC -> shared library -> dlopen"; here NVRTC -> cubin ->
// cudaLibraryLoadData) and keeps it loaded for the life of the context so that every expression is compiled
// once per process.  Real scalars travel as kernel arguments (the POD part of the tree), so
// expressions that differ only in their scalars share a kernel.
#include <dlfcn.h>
#include <string.h>

#include <map>
#include <mutex>
#include <sstream>

#include "lqx_internal.cuh"

// --------------------------------------------------------------------------------------------
// NVRTC, loaded lazily: the library itself keeps no link-time dependency on it
// --------------------------------------------------------------------------------------------
namespace {

typedef struct _nvrtcProgram* nvrtcProgram;
struct Nvrtc {
    void* h = nullptr;
    int (*CreateProgram)(nvrtcProgram*, const char*, const char*, int, const char* const*, const char* const*) = nullptr;
    int (*CompileProgram)(nvrtcProgram, int, const char* const*) = nullptr;
    int (*GetCUBINSize)(nvrtcProgram, size_t*) = nullptr;
    int (*GetCUBIN)(nvrtcProgram, char*) = nullptr;
    int (*GetProgramLogSize)(nvrtcProgram, size_t*) = nullptr;
    int (*GetProgramLog)(nvrtcProgram, char*) = nullptr;
    int (*DestroyProgram)(nvrtcProgram*) = nullptr;
    bool load() {
        if (h) return true;
        const char* names[] = {"libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so.12", "libnvrtc.so"};
        for (const char* n : names) {
            h = dlopen(n, RTLD_NOW | RTLD_LOCAL);
            if (h) break;
        }
        if (!h) return false;
#define LQX_SYM(f) *(void**)(&f) = dlsym(h, "nvrtc" #f)
        LQX_SYM(CreateProgram);
        LQX_SYM(CompileProgram);
        LQX_SYM(GetCUBINSize);
        LQX_SYM(GetCUBIN);
        LQX_SYM(GetProgramLogSize);
        LQX_SYM(GetProgramLog);
        LQX_SYM(DestroyProgram);
#undef LQX_SYM
        return CreateProgram && CompileProgram && GetCUBINSize && GetCUBIN && GetProgramLogSize && GetProgramLog && DestroyProgram;
    }
};
Nvrtc g_nvrtc;

// --------------------------------------------------------------------------------------------
// device prelude of every generated kernel: geometry, blocked-SoA loads/stores (the layout of
// lqx_internal.cuh restated; include/lqx.h documents it) and the site algebra
// --------------------------------------------------------------------------------------------
const char* kPrelude = R"SRC(
struct JGeo { int L[4]; int st[4]; int V; };
template <int N> struct Obj { T re[N], im[N]; };   // N complex numbers in QDP order
// PLAIN: ordinary loads instead of the read-only path -- for the destination of `+=` and for every leaf of a kernel
// whose destination IS one of its leaves (in place, site-local): ld.global.nc is defined only for memory the kernel
// never writes
template <int N, bool PLAIN = kAllPlain>
__device__ __forceinline__ Obj<N> jload(const T* base, int s) {
    constexpr int NREAL = 2 * N, NFULL = NREAL / W;
    T r[NREAL];
    const T* blk = base + (size_t)(s >> 5) * (32 * NREAL);
    const int lane = s & 31;
    const VEC* p = reinterpret_cast<const VEC*>(blk) + lane;
#pragma unroll
    for (int q = 0; q < NFULL; ++q) {
        const VEC v = PLAIN ? p[q * 32] : __ldg(p + q * 32);
        const T* e = reinterpret_cast<const T*>(&v);
#pragma unroll
        for (int k = 0; k < W; ++k) r[q * W + k] = e[k];
    }
    if (NREAL % W != 0) {
        const float2* ph = reinterpret_cast<const float2*>(blk + NFULL * 32 * W) + lane;
        const float2 t = PLAIN ? *ph : __ldg(ph);
        r[NFULL * W] = (T)t.x;
        r[NFULL * W + 1] = (T)t.y;
    }
    Obj<N> o;
#pragma unroll
    for (int i = 0; i < N; ++i) { o.re[i] = r[2 * i]; o.im[i] = r[2 * i + 1]; }
    return o;
}
template <int N>
__device__ __forceinline__ void jstore(T* base, int s, const Obj<N>& o) {
    constexpr int NREAL = 2 * N, NFULL = NREAL / W;
    T r[NREAL];
#pragma unroll
    for (int i = 0; i < N; ++i) { r[2 * i] = o.re[i]; r[2 * i + 1] = o.im[i]; }
    T* blk = base + (size_t)(s >> 5) * (32 * NREAL);
    const int lane = s & 31;
    VEC* p = reinterpret_cast<VEC*>(blk) + lane;
#pragma unroll
    for (int q = 0; q < NFULL; ++q) {
        VEC v;
        T* e = reinterpret_cast<T*>(&v);
#pragma unroll
        for (int k = 0; k < W; ++k) e[k] = r[q * W + k];
        p[q * 32] = v;
    }
    if (NREAL % W != 0) reinterpret_cast<float2*>(blk + NFULL * 32 * W)[lane] = make_float2((float)r[NFULL * W], (float)r[NFULL * W + 1]);
}
template <int N> __device__ __forceinline__ Obj<N> jadd(const Obj<N>& a, const Obj<N>& b) {
    Obj<N> c;
#pragma unroll
    for (int i = 0; i < N; ++i) { c.re[i] = a.re[i] + b.re[i]; c.im[i] = a.im[i] + b.im[i]; }
    return c;
}
template <int N> __device__ __forceinline__ Obj<N> jsub(const Obj<N>& a, const Obj<N>& b) {
    Obj<N> c;
#pragma unroll
    for (int i = 0; i < N; ++i) { c.re[i] = a.re[i] - b.re[i]; c.im[i] = a.im[i] - b.im[i]; }
    return c;
}
template <int N> __device__ __forceinline__ Obj<N> jscale(T k, const Obj<N>& a) {
    Obj<N> c;
#pragma unroll
    for (int i = 0; i < N; ++i) { c.re[i] = k * a.re[i]; c.im[i] = k * a.im[i]; }
    return c;
}
__device__ __forceinline__ Obj<9> jadj(const Obj<9>& a) {   // element (i,j) = index 3*i+j
    Obj<9> c;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) { c.re[3 * i + j] = a.re[3 * j + i]; c.im[3 * i + j] = -a.im[3 * j + i]; }
    return c;
}
// matrix (9) times NV colour vectors (3*NV complex; NV = 3 with the vectors as COLUMNS is matrix*matrix)
__device__ __forceinline__ Obj<9> jmul(const Obj<9>& a, const Obj<9>& b) {
    Obj<9> c;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            T re = a.re[3 * i] * b.re[j], im = a.re[3 * i] * b.im[j];
            re = fma(-a.im[3 * i], b.im[j], re);
            im = fma(a.im[3 * i], b.re[j], im);
#pragma unroll
            for (int k = 1; k < 3; ++k) {
                re = fma(a.re[3 * i + k], b.re[3 * k + j], re);
                im = fma(a.re[3 * i + k], b.im[3 * k + j], im);
                re = fma(-a.im[3 * i + k], b.im[3 * k + j], re);
                im = fma(a.im[3 * i + k], b.re[3 * k + j], im);
            }
            c.re[3 * i + j] = re;
            c.im[3 * i + j] = im;
        }
    return c;
}
// c + a*b with the products accumulated straight into c (what `x + m*y` compiles to)
__device__ __forceinline__ Obj<9> jmac(const Obj<9>& c0, const Obj<9>& a, const Obj<9>& b) {
    Obj<9> c;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            T re = c0.re[3 * i + j], im = c0.im[3 * i + j];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                re = fma(a.re[3 * i + k], b.re[3 * k + j], re);
                im = fma(a.re[3 * i + k], b.im[3 * k + j], im);
                re = fma(-a.im[3 * i + k], b.im[3 * k + j], re);
                im = fma(a.im[3 * i + k], b.re[3 * k + j], im);
            }
            c.re[3 * i + j] = re;
            c.im[3 * i + j] = im;
        }
    return c;
}
template <int NV>
__device__ __forceinline__ Obj<3 * NV> jmacv(const Obj<3 * NV>& w0, const Obj<9>& m, const Obj<3 * NV>& v) {
    Obj<3 * NV> w;
#pragma unroll
    for (int a = 0; a < NV; ++a)
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            T re = w0.re[3 * a + i], im = w0.im[3 * a + i];
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                re = fma(m.re[3 * i + j], v.re[3 * a + j], re);
                im = fma(m.re[3 * i + j], v.im[3 * a + j], im);
                re = fma(-m.im[3 * i + j], v.im[3 * a + j], re);
                im = fma(m.im[3 * i + j], v.re[3 * a + j], im);
            }
            w.re[3 * a + i] = re;
            w.im[3 * a + i] = im;
        }
    return w;
}
__device__ __forceinline__ Obj<1> jtrace(const Obj<9>& a) {
    Obj<1> c;
    c.re[0] = a.re[0] + a.re[4] + a.re[8];
    c.im[0] = a.im[0] + a.im[4] + a.im[8];
    return c;
}
// per-CTA sum of NC doubles per thread -> partials[c * gridDim.x + blockIdx.x] (fixed tree: deterministic)
template <int NC>
__device__ __forceinline__ void jreduce(double (&v)[NC], double* __restrict__ partials) {
    __shared__ double sh[4][NC];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        double t = v[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (lane == 0) sh[warp][c] = t;
    }
    __syncthreads();
    if (threadIdx.x < NC) partials[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = (sh[0][threadIdx.x] + sh[1][threadIdx.x]) + (sh[2][threadIdx.x] + sh[3][threadIdx.x]);
}
template <int NV>
__device__ __forceinline__ Obj<3 * NV> jmulv(const Obj<9>& m, const Obj<3 * NV>& v) {
    Obj<3 * NV> w;
#pragma unroll
    for (int a = 0; a < NV; ++a)
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            T re = m.re[3 * i] * v.re[3 * a], im = m.re[3 * i] * v.im[3 * a];
            re = fma(-m.im[3 * i], v.im[3 * a], re);
            im = fma(m.im[3 * i], v.re[3 * a], im);
#pragma unroll
            for (int j = 1; j < 3; ++j) {
                re = fma(m.re[3 * i + j], v.re[3 * a + j], re);
                im = fma(m.re[3 * i + j], v.im[3 * a + j], im);
                re = fma(-m.im[3 * i + j], v.im[3 * a + j], re);
                im = fma(m.im[3 * i + j], v.re[3 * a + j], im);
            }
            w.re[3 * a + i] = re;
            w.im[3 * a + i] = im;
        }
    return w;
}
)SRC";

}  // namespace

// --------------------------------------------------------------------------------------------
// host: flattened tree -> checked tree -> source
// --------------------------------------------------------------------------------------------
namespace {

struct XNode {
    int op, a, b;      // see lqx_xop
    int child[2];      // indices into the node vector (-1 = none)
    int kind;          // complex numbers per site of the value (lqx_kind)
    int scalar_slot;   // SCALE: index into the scalar argument array
};

struct JitKernel {
    cudaLibrary_t lib;
    cudaKernel_t fn;
};

struct JitCache {
    std::map<std::string, JitKernel> kernels;
};
std::map<lqx_ctx*, JitCache> g_caches;  // per context; emptied by lqx_jit_release (called from lqx_finalize)
std::mutex g_caches_mutex;              // contexts may live on different host threads

// recursive code generation: emits statements into `os`, returns the name of the value's variable.
// A site is a variable holding its index plus the names of its four coordinates, so that a shift is a
// compare-and-select on ONE coordinate (no division), however deeply shifts nest.
struct Site {
    std::string s, x[4];
};
struct Gen {
    const std::vector<XNode>& n;
    std::ostringstream os;
    int tmp = 0, sites = 0;
    explicit Gen(const std::vector<XNode>& nodes) : n(nodes) {}
    // shift(expr, dir, mu)(x) = expr(x + dir*mu^): the operand is evaluated at the neighbour site
    Site shifted(const Site& site, const XNode& x) {
        const std::string k = std::to_string(++sites), mu = std::to_string(x.b);
        Site s2 = site;
        s2.s = "s" + k;
        s2.x[x.b] = "x" + k;
        if (x.a > 0) os << "    const int x" << k << " = " << site.x[x.b] << " + 1 == g.L[" << mu << "] ? 0 : " << site.x[x.b] << " + 1;\n";
        else os << "    const int x" << k << " = " << site.x[x.b] << " == 0 ? g.L[" << mu << "] - 1 : " << site.x[x.b] << " - 1;\n";
        os << "    const int s" << k << " = " << site.s << " + (x" << k << " - " << site.x[x.b] << ") * g.st[" << mu << "];\n";
        return s2;
    }
    // `other + m*y` (the product possibly under shifts) -> one multiply-accumulate into `other`
    bool try_mac(int other, int prod, const Site& site, const std::string& v, const std::string& ty) {
        Site ps = site;
        int pi = prod;
        // only peek: shifts are emitted after the decision
        while (n[pi].op == LQX_X_SHIFT) pi = n[pi].child[0];
        if (n[pi].op != LQX_X_MUL) return false;
        const std::string l = val(other, site);
        for (pi = prod; n[pi].op == LQX_X_SHIFT; pi = n[pi].child[0]) ps = shifted(ps, n[pi]);
        const std::string a = val(n[pi].child[0], ps), b = val(n[pi].child[1], ps);
        if (n[n[pi].child[1]].kind == LQX_COLORMAT) os << "    const " << ty << " " << v << " = jmac(" << l << ", " << a << ", " << b << ");\n";
        else os << "    const " << ty << " " << v << " = jmacv<" << n[pi].kind / 3 << ">(" << l << ", " << a << ", " << b << ");\n";
        return true;
    }
    // the terms of a tree of additions, left to right; a shift of a sum is the sum of the shifted terms
    void collect_terms(int i, const Site& site, std::vector<std::pair<int, Site>>& terms) {
        const XNode& x = n[i];
        if (x.op == LQX_X_ADD) {
            collect_terms(x.child[0], site, terms);
            collect_terms(x.child[1], site, terms);
            return;
        }
        if (x.op == LQX_X_SHIFT) {
            int c = x.child[0];
            while (n[c].op == LQX_X_SHIFT) c = n[c].child[0];
            if (n[c].op == LQX_X_ADD) {
                collect_terms(x.child[0], shifted(site, x), terms);
                return;
            }
        }
        terms.push_back(std::make_pair(i, site));
    }
    // acc + m*y (the product possibly under shifts) as one multiply-accumulate named v; false if term is no product
    bool emit_mac(const std::string& acc, int prod, const Site& site, const std::string& v, const std::string& ty) {
        int pi = prod;
        while (n[pi].op == LQX_X_SHIFT) pi = n[pi].child[0];
        if (n[pi].op != LQX_X_MUL) return false;
        Site ps = site;
        for (pi = prod; n[pi].op == LQX_X_SHIFT; pi = n[pi].child[0]) ps = shifted(ps, n[pi]);
        const std::string a = val(n[pi].child[0], ps), b = val(n[pi].child[1], ps);
        if (n[n[pi].child[1]].kind == LQX_COLORMAT) os << "    const " << ty << " " << v << " = jmac(" << acc << ", " << a << ", " << b << ");\n";
        else os << "    const " << ty << " " << v << " = jmacv<" << n[pi].kind / 3 << ">(" << acc << ", " << a << ", " << b << ");\n";
        return true;
    }
    std::string val(int i, const Site& site) {
        const XNode& x = n[i];
        const std::string ty = "Obj<" + std::to_string(x.kind) + ">";
        if (x.op == LQX_X_SHIFT) return val(x.child[0], shifted(site, x));
        std::string v = "v" + std::to_string(tmp++);
        switch (x.op) {
            case LQX_X_LEAF:
                os << "    const " << ty << " " << v << " = jload<" << x.kind << ">(p" << x.a << ", " << site.s << ");\n";
                break;
            case LQX_X_ADJ: {
                std::string c = val(x.child[0], site);
                os << "    const " << ty << " " << v << " = jadj(" << c << ");\n";
                break;
            }
            case LQX_X_MUL: {
                std::string l = val(x.child[0], site), r = val(x.child[1], site);
                if (n[x.child[1]].kind == LQX_COLORMAT) os << "    const " << ty << " " << v << " = jmul(" << l << ", " << r << ");\n";
                else os << "    const " << ty << " " << v << " = jmulv<" << x.kind / 3 << ">(" << l << ", " << r << ");\n";
                break;
            }
            case LQX_X_ADD:
            case LQX_X_SUB: {
                if (x.op == LQX_X_ADD) {
                    // a sum of three or more terms is evaluated as ONE accumulation chain in the order written
                    // (t0 + t1 + t2 ... ; products become multiply-accumulates): no partial sums are kept alive
                    // beside the accumulator, which is what lets the hop run at six CTAs per SM
                    std::vector<std::pair<int, Site>> terms;
                    collect_terms(i, site, terms);
                    if (terms.size() > 2) {
                        std::string acc = val(terms[0].first, terms[0].second);
                        for (size_t t = 1; t < terms.size(); ++t) {
                            const std::string name = t + 1 == terms.size() ? v : "v" + std::to_string(tmp++);
                            if (!emit_mac(acc, terms[t].first, terms[t].second, name, ty)) {
                                const std::string r = val(terms[t].first, terms[t].second);
                                os << "    const " << ty << " " << name << " = jadd(" << acc << ", " << r << ");\n";
                            }
                            acc = name;
                        }
                        break;
                    }
                }
                if (x.op == LQX_X_ADD && (try_mac(x.child[0], x.child[1], site, v, ty) || try_mac(x.child[1], x.child[0], site, v, ty))) break;
                std::string l = val(x.child[0], site), r = val(x.child[1], site);
                os << "    const " << ty << " " << v << " = " << (x.op == LQX_X_ADD ? "jadd" : "jsub") << "(" << l << ", " << r << ");\n";
                break;
            }
            case LQX_X_TRACE: {
                std::string c = val(x.child[0], site);
                os << "    const " << ty << " " << v << " = jtrace(" << c << ");\n";
                break;
            }
            case LQX_X_SCALE: {
                std::string c = val(x.child[0], site);
                os << "    const " << ty << " " << v << " = jscale(k" << x.scalar_slot << ", " << c << ");\n";
                break;
            }
        }
        return v;
    }
};

int build_tree(lqx_ctx* ctx, const lqx_xnode* nodes, int nnodes, const lqx_field* const* leaves, int nleaves,
               std::vector<XNode>& out, std::vector<double>& scalars, std::vector<bool>& leaf_shifted) {
    std::vector<int> stack;
    out.clear();
    for (int i = 0; i < nnodes; ++i) {
        XNode x;
        x.op = nodes[i].op;
        x.a = nodes[i].a;
        x.b = nodes[i].b;
        x.child[0] = x.child[1] = -1;
        x.scalar_slot = -1;
        x.kind = 0;
        auto pop = [&]() {
            int t = stack.back();
            stack.pop_back();
            return t;
        };
        switch (x.op) {
            case LQX_X_LEAF:
                if (x.a < 0 || x.a >= nleaves) return lqx_fail(ctx, LQX_EINVAL, "expr: leaf index out of range");
                x.kind = (int)leaves[x.a]->kind;
                break;
            case LQX_X_ADJ:
                if (stack.empty()) return lqx_fail(ctx, LQX_EINVAL, "expr: adj without operand");
                x.child[0] = pop();
                if (out[x.child[0]].kind != LQX_COLORMAT) return lqx_fail(ctx, LQX_ETYPE, "expr: adj wants a colour matrix");
                x.kind = LQX_COLORMAT;
                break;
            case LQX_X_TRACE:
                if (stack.empty()) return lqx_fail(ctx, LQX_EINVAL, "expr: trace without operand");
                x.child[0] = pop();
                if (out[x.child[0]].kind != LQX_COLORMAT) return lqx_fail(ctx, LQX_ETYPE, "expr: trace wants a colour matrix");
                x.kind = LQX_COMPLEX;
                break;
            case LQX_X_MUL:
            case LQX_X_ADD:
            case LQX_X_SUB: {
                if (stack.size() < 2) return lqx_fail(ctx, LQX_EINVAL, "expr: binary operator without two operands");
                x.child[1] = pop();
                x.child[0] = pop();
                const int kl = out[x.child[0]].kind, kr = out[x.child[1]].kind;
                if (x.op == LQX_X_MUL) {
                    if (kl != LQX_COLORMAT || kr == LQX_COMPLEX) return lqx_fail(ctx, LQX_ETYPE, "expr: '*' is matrix*matrix or matrix*vector");
                    x.kind = kr;
                } else {
                    if (kl != kr) return lqx_fail(ctx, LQX_ETYPE, "expr: '+'/'-' operands differ in kind");
                    x.kind = kl;
                }
                break;
            }
            case LQX_X_SCALE:
                if (stack.empty()) return lqx_fail(ctx, LQX_EINVAL, "expr: scale without operand");
                x.child[0] = pop();
                x.kind = out[x.child[0]].kind;
                x.scalar_slot = (int)scalars.size();
                scalars.push_back(nodes[i].s);
                break;
            case LQX_X_SHIFT:
                if (stack.empty()) return lqx_fail(ctx, LQX_EINVAL, "expr: shift without operand");
                if ((x.a != 1 && x.a != -1) || x.b < 0 || x.b > 3) return lqx_fail(ctx, LQX_EINVAL, "expr: shift dir/mu");
                x.child[0] = pop();
                x.kind = out[x.child[0]].kind;
                break;
            default:
                return lqx_fail(ctx, LQX_EINVAL, "expr: unknown operator");
        }
        out.push_back(x);
        stack.push_back((int)out.size() - 1);
    }
    if (stack.size() != 1) return lqx_fail(ctx, LQX_EINVAL, "expr: the postfix sequence does not reduce to one value");
    // which leaves are read through a shift (they must not alias the destination)
    leaf_shifted.assign(nleaves, false);
    std::vector<std::pair<int, bool>> todo(1, std::make_pair(stack[0], false));
    while (!todo.empty()) {
        auto [i, sh] = todo.back();
        todo.pop_back();
        const XNode& x = out[i];
        if (x.op == LQX_X_LEAF && sh) leaf_shifted[x.a] = true;
        for (int c = 0; c < 2; ++c)
            if (x.child[c] >= 0) todo.push_back(std::make_pair(x.child[c], sh || x.op == LQX_X_SHIFT));
    }
    return LQX_OK;
}

// Estimate of the reals a thread holds at the widest point of the evaluation (operands are evaluated left to
// right, a sum is one accumulation chain): picks the CTAs-per-SM bound of the generated kernel, so that a small
// expression (the hop: accumulator + one matrix + one fermion) runs at six CTAs per SM and a product of
// products (the plaquette: four matrices and an accumulator) is not forced to spill.
static void live_terms(const std::vector<XNode>& n, int i, std::vector<int>& terms) {
    if (n[i].op == LQX_X_ADD) {
        live_terms(n, n[i].child[0], terms);
        live_terms(n, n[i].child[1], terms);
        return;
    }
    if (n[i].op == LQX_X_SHIFT) {
        int c = n[i].child[0];
        while (n[c].op == LQX_X_SHIFT) c = n[c].child[0];
        if (n[c].op == LQX_X_ADD) {
            live_terms(n, c, terms);
            return;
        }
    }
    terms.push_back(i);
}
static int live_reals(const std::vector<XNode>& n, int i) {
    const XNode& x = n[i];
    const int sz = 2 * x.kind;
    switch (x.op) {
        case LQX_X_LEAF: return sz;
        case LQX_X_MUL: {
            const int l = live_reals(n, x.child[0]), r = live_reals(n, x.child[1]);
            const int sl = 2 * n[x.child[0]].kind, sr = 2 * n[x.child[1]].kind;
            return std::max(std::max(l, sl + r), sl + sr + sz);
        }
        case LQX_X_SUB: return std::max(live_reals(n, x.child[0]), sz + live_reals(n, x.child[1]));
        case LQX_X_ADD: {
            std::vector<int> terms;
            live_terms(n, i, terms);
            int m = live_reals(n, terms[0]);
            for (size_t t = 1; t < terms.size(); ++t) {
                int p = terms[t];
                while (n[p].op == LQX_X_SHIFT) p = n[p].child[0];
                if (n[p].op == LQX_X_MUL) {  // multiply-accumulate: the product has no result of its own
                    const int sl = 2 * n[n[p].child[0]].kind, sr = 2 * n[n[p].child[1]].kind;
                    m = std::max(m, sz + std::max(std::max(live_reals(n, n[p].child[0]), sl + live_reals(n, n[p].child[1])), sl + sr));
                } else {
                    m = std::max(m, sz + live_reals(n, terms[t]));
                }
            }
            return m;
        }
        default: return live_reals(n, x.child[0]);  // adj, shift, scale, trace
    }
}

// reduce: 0 = dst (=|+=) expr ; 1 = norm2(expr) ; 2 = sum(expr).  For the reductions every thread walks a
// grid-stride loop of sites with fp64 accumulators and the CTA leaves one partial per component.
std::string make_source(const std::vector<XNode>& tree, int nleaves, int nscalars, int dst_kind, bool f32, bool accumulate,
                        int reduce, bool inplace) {
    std::ostringstream src;
    if (f32) src << "typedef float T;\ntypedef float4 VEC;\nconstexpr int W = 4;\n";
    else src << "typedef double T;\ntypedef double2 VEC;\nconstexpr int W = 2;\n";
    src << "constexpr bool kAllPlain = " << (inplace ? "true" : "false") << ";\n";
    src << kPrelude;
    // register budget from the estimated live reals (+ fp64 reduction accumulators, + 16 for indices and
    // pointers): at most six CTAs of 128 threads per SM (85 registers) in fp32 and three (170) in fp64, at least two
    const int nacc = reduce == 1 ? 1 : (reduce == 2 ? 2 * dst_kind : 0);
    const int regs = live_reals(tree, (int)tree.size() - 1) * (f32 ? 1 : 2) + 2 * nacc + 16;
    const int min_blocks = std::max(2, std::min(f32 ? 6 : 3, 65536 / (128 * regs)));
    src << "extern \"C\" __global__ void __launch_bounds__(128, " << min_blocks << ") lqx_jit(const JGeo g";
    for (int k = 0; k < nscalars; ++k) src << ", const T k" << k;
    for (int l = 0; l < nleaves; ++l) src << (inplace ? ", const T* p" : ", const T* __restrict__ p") << l;
    const int nc = reduce == 1 ? 1 : 2 * dst_kind;
    if (reduce) {
        src << ", double* __restrict__ partials) {\n    double acc[" << nc << "];\n";
        src << "#pragma unroll\n    for (int c = 0; c < " << nc << "; ++c) acc[c] = 0.0;\n";
        src << "    for (int s0 = blockIdx.x * blockDim.x + threadIdx.x; s0 < g.V; s0 += gridDim.x * blockDim.x) {\n";
    } else {
        src << ", T* dst) {\n    const int s0 = blockIdx.x * blockDim.x + threadIdx.x;\n    if (s0 >= g.V) return;\n";
    }
    src << "    const int x0_0 = s0 % g.L[0], q1 = s0 / g.L[0];\n    const int x0_1 = q1 % g.L[1], q2 = q1 / g.L[1];\n"
           "    const int x0_2 = q2 % g.L[2], x0_3 = q2 / g.L[2];\n";
    Gen gen(tree);
    Site origin;
    origin.s = "s0";
    for (int d = 0; d < 4; ++d) origin.x[d] = "x0_" + std::to_string(d);
    const std::string r = gen.val((int)tree.size() - 1, origin);
    src << gen.os.str();
    if (reduce == 1) {
        src << "#pragma unroll\n    for (int i = 0; i < " << dst_kind << "; ++i) {\n        acc[0] = fma((double)" << r << ".re[i], (double)" << r
            << ".re[i], acc[0]);\n        acc[0] = fma((double)" << r << ".im[i], (double)" << r << ".im[i], acc[0]);\n    }\n    }\n";
        src << "    jreduce<1>(acc, partials);\n";
    } else if (reduce == 2) {
        src << "#pragma unroll\n    for (int i = 0; i < " << dst_kind << "; ++i) {\n        acc[2 * i] += (double)" << r
            << ".re[i];\n        acc[2 * i + 1] += (double)" << r << ".im[i];\n    }\n    }\n";
        src << "    jreduce<" << nc << ">(acc, partials);\n";
    } else if (accumulate) {
        src << "    jstore<" << dst_kind << ">(dst, s0, jadd(jload<" << dst_kind << ", true>(dst, s0), " << r << "));\n";
    } else {
        src << "    jstore<" << dst_kind << ">(dst, s0, " << r << ");\n";
    }
    src << "}\n";
    return src.str();
}

int compile(lqx_ctx* ctx, const std::string& source, JitKernel* out) {
    if (!g_nvrtc.load()) return lqx_fail(ctx, LQX_ECUDA, "expr: libnvrtc.so.12 could not be loaded");
    nvrtcProgram prog;
    if (g_nvrtc.CreateProgram(&prog, source.c_str(), "lqx_jit.cu", 0, nullptr, nullptr) != 0) return lqx_fail(ctx, LQX_ECUDA, "nvrtcCreateProgram");
    const char* opts[] = {"--gpu-architecture=sm_100a", "-std=c++17", "-lineinfo"};
    const int rc = g_nvrtc.CompileProgram(prog, 3, opts);
    if (rc != 0) {
        size_t n = 0;
        g_nvrtc.GetProgramLogSize(prog, &n);
        std::string log(n, '\0');
        if (n) g_nvrtc.GetProgramLog(prog, &log[0]);
        g_nvrtc.DestroyProgram(&prog);
        ctx->last_error = "expr: NVRTC compilation failed: " + log.substr(0, 2000);
        return LQX_ECUDA;
    }
    size_t n = 0;
    g_nvrtc.GetCUBINSize(prog, &n);
    std::vector<char> cubin(n);
    g_nvrtc.GetCUBIN(prog, cubin.data());
    g_nvrtc.DestroyProgram(&prog);
    LQX_CUDA(ctx, cudaLibraryLoadData(&out->lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0));
    LQX_CUDA(ctx, cudaLibraryGetKernel(&out->fn, out->lib, "lqx_jit"));
    return LQX_OK;
}

}  // namespace

void lqx_jit_release(lqx_ctx* ctx) {
    std::lock_guard<std::mutex> lock(g_caches_mutex);
    auto it = g_caches.find(ctx);
    if (it == g_caches.end()) return;
    for (auto& kv : it->second.kernels) cudaLibraryUnload(kv.second.lib);
    g_caches.erase(it);
}

extern "C" int lqx_expr_cache_size(const lqx_ctx* ctx) {
    if (!ctx) return LQX_EINVAL;
    std::lock_guard<std::mutex> lock(g_caches_mutex);
    auto it = g_caches.find(const_cast<lqx_ctx*>(ctx));
    return it == g_caches.end() ? 0 : (int)it->second.kernels.size();
}

extern "C" int lqx_expr_source(lqx_ctx* ctx, lqx_kind dst_kind, lqx_prec prec, int accumulate, const lqx_xnode* nodes, int nnodes,
                               const lqx_kind* leaf_kinds, int nleaves, char* buf, size_t buflen) {
    if (!nodes || nnodes <= 0 || !buf || buflen == 0 || (nleaves > 0 && !leaf_kinds)) return LQX_EINVAL;  // ctx may be NULL
    std::vector<lqx_field> fake(nleaves);
    std::vector<const lqx_field*> leaves(nleaves);
    for (int l = 0; l < nleaves; ++l) {
        fake[l].ctx = ctx;
        fake[l].kind = leaf_kinds[l];
        fake[l].prec = prec;
        fake[l].data = nullptr;
        fake[l].owned = false;
        leaves[l] = &fake[l];
    }
    std::vector<XNode> tree;
    std::vector<double> scalars;
    std::vector<bool> shifted;
    int rc = build_tree(ctx, nodes, nnodes, leaves.data(), nleaves, tree, scalars, shifted);
    if (rc) return rc;
    if (tree.back().kind != (int)dst_kind) return lqx_fail(ctx, LQX_ETYPE, "expr: destination kind differs from the expression's");
    const int reduce = accumulate >= 2 ? accumulate - 1 : 0;  // 2, 3: the kernels of lqx_expr_reduce (norm2, sum)
    const std::string src = make_source(tree, nleaves, (int)scalars.size(), (int)dst_kind, prec == LQX_F32, accumulate == 1, reduce, false);
    strncpy(buf, src.c_str(), buflen - 1);
    buf[buflen - 1] = '\0';
    return (int)src.size();
}

// shared by lqx_expr_eval (reduce = 0, dst != NULL) and lqx_expr_reduce (reduce = 1 norm2 / 2 sum, dst == NULL)
static int run_expr(lqx_ctx* ctx, lqx_prec prec, lqx_field* dst, int accumulate, int reduce, const lqx_xnode* nodes, int nnodes,
                    const lqx_field* const* leaves, int nleaves, double* out, int* out_count) {
    if (nleaves > 16) return lqx_fail(ctx, LQX_EINVAL, "expr: at most 16 leaves");
    for (int l = 0; l < nleaves; ++l) {
        if (!leaves[l]) return LQX_EINVAL;
        if (leaves[l]->ctx != ctx) return lqx_fail(ctx, LQX_EGEOM, "expr: leaves belong to different contexts");
        if (leaves[l]->prec != prec) return lqx_fail(ctx, LQX_ETYPE, "expr: mixed precision");
    }
    std::vector<XNode> tree;
    std::vector<double> scalars;
    std::vector<bool> shifted;
    int rc = build_tree(ctx, nodes, nnodes, leaves, nleaves, tree, scalars, shifted);
    if (rc) return rc;
    if (scalars.size() > 16) return lqx_fail(ctx, LQX_EINVAL, "expr: at most 16 scalars");
    const int kind = tree.back().kind;
    bool inplace = false;
    if (dst) {
        if (kind != (int)dst->kind) return lqx_fail(ctx, LQX_ETYPE, "expr: destination kind differs from the expression's");
        for (int l = 0; l < nleaves; ++l) {
            if (shifted[l] && lqx_same(dst, leaves[l])) return lqx_fail(ctx, LQX_EALIAS, "expr: destination is read through a shift");
            if (lqx_identical(dst, leaves[l])) inplace = true;  // site-local use of the destination (A21)
            else if (lqx_same(dst, leaves[l])) return lqx_fail(ctx, LQX_EALIAS, "expr: destination partially overlaps a leaf");
        }
    }
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const bool f32 = prec == LQX_F32;
    const std::string src = make_source(tree, nleaves, (int)scalars.size(), kind, f32, accumulate != 0, reduce, inplace);
    cudaKernel_t fn;
    {
        std::lock_guard<std::mutex> lock(g_caches_mutex);
        JitCache& cache = g_caches[ctx];
        auto it = cache.kernels.find(src);
        if (it == cache.kernels.end()) {
            JitKernel k;
            rc = compile(ctx, src, &k);
            if (rc) return rc;
            it = cache.kernels.insert(std::make_pair(src, k)).first;
        }
        fn = it->second.fn;
    }
    // arguments: geometry, scalars (rounded once to the field precision, reading A10), leaf pointers, destination
    struct JGeo {
        int L[4], st[4], V;
    } jg;
    for (int d = 0; d < 4; ++d) {
        jg.L[d] = ctx->geo.L[d];
        jg.st[d] = ctx->geo.stride_site[d];
    }
    jg.V = ctx->geo.V;
    float kf[16];
    double kd[16];
    const void* ptrs[16];
    void* args[1 + 16 + 16 + 1];
    int na = 0;
    args[na++] = &jg;
    for (size_t k = 0; k < scalars.size(); ++k) {
        kf[k] = (float)scalars[k];
        kd[k] = scalars[k];
        args[na++] = f32 ? (void*)&kf[k] : (void*)&kd[k];
    }
    for (int l = 0; l < nleaves; ++l) {
        ptrs[l] = leaves[l]->data;
        args[na++] = &ptrs[l];
    }
    int grid = (ctx->geo.V + 127) / 128;
    void* dptr = nullptr;
    const int nc = reduce == 1 ? 1 : 2 * kind;
    if (reduce) {
        grid = std::max(1, std::min(grid, ctx->num_sms * 16));  // fixed function of V: deterministic summation tree
        rc = lqx_ensure_partials(ctx, (size_t)grid * nc);
        if (rc) return rc;
        dptr = ctx->d_partials;
    } else {
        dptr = dst->data;
    }
    args[na++] = &dptr;
    {
        LqxTimed timed(ctx, reduce ? LQX_K_REDUCE : LQX_K_CATALOGUE);
        LQX_CUDA(ctx, cudaLaunchKernel((const void*)fn, dim3(grid), dim3(128), args, 0, ctx->stream));
    }
    ctx->launches++;
    if (!reduce) return LQX_OK;
    rc = lqx_sum_partials(ctx, grid, nc, ctx->h_result);
    if (rc) return rc;
    if (out_count) *out_count = nc;
    return lqx_fetch_result(ctx, nc, out);
}

extern "C" int lqx_expr_eval(lqx_field* dst, int accumulate, const lqx_xnode* nodes, int nnodes, const lqx_field* const* leaves,
                             int nleaves) {
    if (!dst || !nodes || nnodes <= 0 || nleaves < 0 || (nleaves > 0 && !leaves)) return LQX_EINVAL;
    return run_expr(dst->ctx, dst->prec, dst, accumulate, 0, nodes, nnodes, leaves, nleaves, nullptr, nullptr);
}

extern "C" int lqx_expr_reduce(int what, const lqx_xnode* nodes, int nnodes, const lqx_field* const* leaves, int nleaves,
                               double* out, int* out_count) {
    if (!nodes || nnodes <= 0 || nleaves <= 0 || !leaves || !leaves[0] || !out) return LQX_EINVAL;
    lqx_ctx* ctx = leaves[0]->ctx;
    if (what != LQX_R_NORM2 && what != LQX_R_SUM) return lqx_fail(ctx, LQX_EINVAL, "expr_reduce: unknown reduction");
    return run_expr(ctx, leaves[0]->prec, nullptr, 0, what, nodes, nnodes, leaves, nleaves, out, out_count);
}
