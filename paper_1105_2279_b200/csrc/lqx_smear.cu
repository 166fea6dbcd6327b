// lqx staple sum + smear step kernels (BASELINE.json configs[0],[2],[3]):
//   S_mu(x)  = sum_{nu!=mu} U_nu(x) U_mu(x+nu^) adj(U_nu(x+mu^)) + adj(U_nu(x-nu^)) U_mu(x-nu^) U_nu(x-nu^+mu^)
//   U'_mu(x) = c0 U_mu(x) + c1 S_mu(x),   c0 = 1-alpha, c1 = alpha/6
// One thread evaluates the whole expression of its site; the shifted operands
// are read at periodic neighbours computed in-kernel.  Variants of the same
// literal 48-product evaluation, selected by the context option "smear_variant":
//   1  k_smear_gather : mu outer / nu inner as run-time loops, one accumulator (also the staple_sum entry)
//   3  k_smear_rolled : same order, neighbour indices in shared memory, U_mu(x) not held, register cap
//                       that allows three 256-thread (six 128-thread) CTAs per SM in fp32  [default]
//   4  k_smear_mu4    : four threads per site (one per link) on 64/128-site tiles whose operands fit L1
// Tried and dropped: full unrolling of mu, nu (255 registers + spills), L1 prefetch
// of the next staple's operands (4.3 ms: the L1 request path is the busy unit), nu-outer with four
// accumulators (60 instead of 76 operand fetches, but 168 registers: 3.5 ms).
#include "lqx_smear.cuh"

#include <type_traits>

namespace {

// variant 1: mu outer / nu inner as run-time loops; every staple is a chain of two products kept in
// registers (48 products per site).
// PLAQ: the plaquette of the INPUT field is accumulated on the way:
//   Re tr[U_mu U_nu(x+mu) adj(U_mu(x+nu)) adj(U_nu)] = Re tr[U_mu(x) adj(upper staple_{mu,nu}(x))], mu<nu.
// only_mu >= 0: write the bare staple sum of that direction into out.u[0] (diagnostic entry).
// ---------------------------------------------------------------------------------------------
template <typename T, bool PLAQ, typename MAP>
__global__ void __launch_bounds__(MAP::THREADS) k_smear_gather(const __grid_constant__ Geo g, const __grid_constant__ TileMap tm,
                                                               const __grid_constant__ Links<T> u, const __grid_constant__ LinksOut<T> out,
                                                               T c0, T c1, int only_mu, double* __restrict__ partials,
                                                               unsigned int* ticket, double* __restrict__ red_out) {
    int x[4], s;
    double p[1] = {0.0};
    if (MAP::site(g, tm, x, s)) {
        T pl = T(0);
        const int mu_lo = only_mu >= 0 ? only_mu : 0, mu_hi = only_mu >= 0 ? only_mu + 1 : 4;
#pragma unroll 1
        for (int mu = mu_lo; mu < mu_hi; ++mu) {
            const int xpmu = nbr_fwd(g, s, x, mu);
            const Mat3<T> umu = load_mat(u.u[mu], s);
            Mat3<T> acc = zero_mat<T>();
#pragma unroll 1
            for (int nu = 0; nu < 4; ++nu) {
                if (nu == mu) continue;
                const int xpnu = nbr_fwd(g, s, x, nu);
                const int xmnu = nbr_bwd(g, s, x, nu);
                // x - nu^ + mu^ : step forward in mu from xmnu (coordinates differ from x only in nu)
                const int xmnupmu = xmnu + (xpmu - s);
                {
                    const Mat3<T> t = mul_nn(load_mat(u.u[nu], s), load_mat(u.u[mu], xpnu));
                    if (PLAQ && mu < nu) {
                        const Mat3<T> up = mul_na(t, load_mat(u.u[nu], xpmu));
                        pl += re_tr_na(umu, up);
#pragma unroll
                        for (int i = 0; i < 3; ++i)
#pragma unroll
                            for (int j = 0; j < 3; ++j) {
                                acc.re[i][j] += up.re[i][j];
                                acc.im[i][j] += up.im[i][j];
                            }
                    } else {
                        mac_na(acc, t, load_mat(u.u[nu], xpmu));
                    }
                }
                {
                    const Mat3<T> t = mul_an(load_mat(u.u[nu], xmnu), load_mat(u.u[mu], xmnu));
                    mac_nn(acc, t, load_mat(u.u[nu], xmnupmu));
                }
            }
            if (only_mu >= 0) {
                store_mat(out.u[0], s, acc);
            } else {
                Mat3<T> r;
#pragma unroll
                for (int i = 0; i < 3; ++i)
#pragma unroll
                    for (int j = 0; j < 3; ++j) {
                        r.re[i][j] = fma(c1, acc.re[i][j], c0 * umu.re[i][j]);
                        r.im[i][j] = fma(c1, acc.im[i][j], c0 * umu.im[i][j]);
                    }
                store_mat(out.u[mu], s, r);
            }
        }
        p[0] = (double)pl;
    }
    if (PLAQ) block_reduce_partial<1>(p, partials);
}


template <typename T>
__device__ __forceinline__ void add_to(Mat3<T>& acc, const Mat3<T>& m) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            acc.re[i][j] += m.re[i][j];
            acc.im[i][j] += m.im[i][j];
        }
}
template <typename T>
__device__ __forceinline__ Mat3<T> smear_update(T c0, T c1, const Mat3<T>& umu, const Mat3<T>& acc) {
    Mat3<T> r;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            r.re[i][j] = fma(c1, acc.re[i][j], c0 * umu.re[i][j]);
            r.im[i][j] = fma(c1, acc.im[i][j], c0 * umu.im[i][j]);
        }
    return r;
}

// variant 3: the literal evaluation with the loops kept rolled (so that only one staple's operands are
// live: 80 registers, three 256-thread CTAs per SM in fp32), the eight neighbour site indices of the
// thread parked in shared memory and looked up by the run-time direction, and U_mu(x) fetched only
// when it is needed instead of being held across the nu loop.  Per link: the three upper staples (nu
// DEscending, the order every variant sums in), then the three lower staples, then U_mu(x) is loaded
// once for the update -- and for the plaquette of the input field, which costs no load of its own:
// every staple of link mu closes one plaquette with U_mu(x) (an upper one P_munu(x), a lower one
// P_munu(x-nu^)), and over the whole periodic lattice every plaquette is met four times, so
//   sum_x sum_{mu<nu} Re tr P_munu(x) = (1/4) sum_x sum_mu Re tr[U_mu(x) adj(S_mu(x))]
// (SURVEY 8(c) staple pin; exact for the GLOBAL sum only, which is all a launch reports: the ranged
// launches of the streamed host path run with PLAQ = false).  An extra trace after the nu > mu staples, as before, re-read
// U_mu(x) for three links: +4 % on a kernel that is bound by the L1 data pipe.
template <typename T, bool PLAQ, typename MAP, int MINB>
__global__ void __launch_bounds__(MAP::THREADS, MINB) k_smear_rolled(const __grid_constant__ Geo g, const __grid_constant__ TileMap tm,
                                                                     const __grid_constant__ Links<T> u, const __grid_constant__ LinksOut<T> out,
                                                                     T c0, T c1, double* __restrict__ partials, unsigned int* ticket,
                                                                     double* __restrict__ red_out) {
    __shared__ int nb[8][MAP::THREADS];  // [0..3] x+d^, [4..7] x-d^
    int x[4], s;
    double p[1] = {0.0};
    const int tid = threadIdx.x;
    if (MAP::site(g, tm, x, s)) {
#pragma unroll
        for (int d = 0; d < 4; ++d) {
            nb[d][tid] = (x[d] + 1 == g.L[d]) ? s - (g.L[d] - 1) * g.stride_site[d] : s + g.stride_site[d];
            nb[4 + d][tid] = (x[d] == 0) ? s + (g.L[d] - 1) * g.stride_site[d] : s - g.stride_site[d];
        }
        T pl = T(0);
#pragma unroll 1
        for (int mu = 0; mu < 4; ++mu) {
            const T* __restrict__ umu_p = u.u[mu];
            const int xpmu = nb[mu][tid];
            Mat3<T> acc = zero_mat<T>();
#pragma unroll 1
            for (int nu = 3; nu >= 0; --nu) {  // upper: U_nu(x) U_mu(x+nu^) adj(U_nu(x+mu^))
                if (nu == mu) continue;
                const T* __restrict__ unu_p = u.u[nu];
                const Mat3<T> t = mul_nn(load_mat(unu_p, s), load_mat(umu_p, nb[nu][tid]));
                mac_na(acc, t, load_mat(unu_p, xpmu));
            }
#pragma unroll 1
            for (int nu = 0; nu < 4; ++nu) {  // lower: adj(U_nu(x-nu^)) U_mu(x-nu^) U_nu(x-nu^+mu^)
                if (nu == mu) continue;
                const T* __restrict__ unu_p = u.u[nu];
                const int xmnu = nb[4 + nu][tid];
                const Mat3<T> t = mul_an(load_mat(unu_p, xmnu), load_mat(umu_p, xmnu));
                mac_nn(acc, t, load_mat(unu_p, xmnu + (xpmu - s)));
            }
            const Mat3<T> umu = load_mat(umu_p, s);
            if (PLAQ) pl += re_tr_na(umu, acc);
            store_mat_cs(out.u[mu], s, smear_update(c0, c1, umu, acc));
        }
        p[0] = 0.25 * (double)pl;
    }
    if (PLAQ) block_reduce_partial<1>(p, partials);
}

// variant 2: shared-corner evaluation.  With Q = U_nu(x) U_mu(x+nu^) the thread of site x
// gets, for the ordered pair (mu, nu), the upper staple of ITS link mu, Q adj(U_nu(x+mu^)), and the lower
// staple of link nu at the neighbour x+mu^, adj(U_mu(x)) Q -- 36 products per site instead of 48 and 16
// distinct operand matrices instead of 44.  The lower staples travel one site in direction mu through
// shared memory: slot[site][link] (one 3x3 matrix each, laid out [link][chunk][site] so that neighbouring
// sites are neighbouring 16-byte words: conflict-free even for the x-shifted site).  Phase mu = 0..3:
//   (a) every thread: its three pairs (mu, nu != mu): upper staples into a register accumulator, lower
//       staples added into slot[x+mu^][nu] if x+mu^ is inside the CTA's tile;
//   (b) the lower staples that ENTER the tile through its low-mu face come from sites of the neighbouring
//       tile: 3*THREADS/T_mu work items (face site, nu), spread evenly over the CTA's threads, each the
//       literal two products adj(U_mu(y)) U_nu(y) U_mu(y+nu^), y = x-mu^, added into slot[x][nu];
//   (c) the thread adds its accumulator into slot[x][mu];  __syncthreads().
// In one phase every slot[.][link != mu] receives exactly one lower staple "from direction mu" (from the
// in-tile neighbour or from a halo item) and slot[.][mu] only its owner's uppers, so the read-modify-
// writes never collide and the summation order is fixed: results are bit-reproducible.
// After the four phases U'_mu(x) = c0 U_mu(x) + c1 slot[x][mu].
template <typename T, int NT>
struct Slots {
    typedef typename Vec128<T>::type V;
    static constexpr int W = Vec128<T>::W, NFULL = 18 / W;
    T* base;
    __device__ __forceinline__ T* link(int l) const { return base + l * (18 * NT); }
    __device__ __forceinline__ void zero(int site, int l) const {
        T* b = link(l);
        const T z[4] = {T(0), T(0), T(0), T(0)};
#pragma unroll
        for (int q = 0; q < NFULL; ++q) reinterpret_cast<V*>(b + q * W * NT)[site] = pack(z);
        if (18 % W != 0) reinterpret_cast<float2*>(b + NFULL * W * NT)[site] = make_float2(0.f, 0.f);
    }
    __device__ __forceinline__ void add(int site, int l, const Mat3<T>& m) const {
        T r[18];
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                r[2 * (3 * i + j)] = m.re[i][j];
                r[2 * (3 * i + j) + 1] = m.im[i][j];
            }
        T* b = link(l);
#pragma unroll
        for (int q = 0; q < NFULL; ++q) {
            V* p = reinterpret_cast<V*>(b + q * W * NT) + site;
            T o[W];
            unpack(*p, o);
#pragma unroll
            for (int k = 0; k < W; ++k) o[k] += r[q * W + k];
            *p = pack(o);
        }
        if (18 % W != 0) {
            float2* p = reinterpret_cast<float2*>(b + NFULL * W * NT) + site;
            float2 o = *p;
            o.x += (float)r[NFULL * W];
            o.y += (float)r[NFULL * W + 1];
            *p = o;
        }
    }
    __device__ __forceinline__ Mat3<T> get(int site, int l) const {
        T r[18];
        const T* b = link(l);
#pragma unroll
        for (int q = 0; q < NFULL; ++q) unpack(reinterpret_cast<const V*>(b + q * W * NT)[site], &r[q * W]);
        if (18 % W != 0) {
            const float2 o = reinterpret_cast<const float2*>(b + NFULL * W * NT)[site];
            r[NFULL * W] = (T)o.x;
            r[NFULL * W + 1] = (T)o.y;
        }
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
};

template <typename T, bool PLAQ, typename MAP, int MINB>
__global__ void __launch_bounds__(MAP::THREADS, MINB) k_smear_shared(const __grid_constant__ Geo g, const __grid_constant__ TileMap tm,
                                                                     const __grid_constant__ Links<T> u, const __grid_constant__ LinksOut<T> out,
                                                                     T c0, T c1, double* __restrict__ partials) {
    constexpr int NT = MAP::THREADS;
    constexpr int T0 = MAP::T0, T1 = MAP::T1, T2 = MAP::T2, T3 = MAP::T3;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Slots<T, NT> slots;
    slots.base = reinterpret_cast<T*>(smem_raw);
    int(*nb)[NT] = reinterpret_cast<int(*)[NT]>(smem_raw + sizeof(T) * 4 * 18 * NT);  // [0..3] x+d^
    int x[4], s;
    MAP::site(g, tm, x, s);  // tiles always cover whole sites
    const int tid = threadIdx.x;
    const int l[4] = {tid % T0, (tid / T0) % T1, (tid / (T0 * T1)) % T2, tid / (T0 * T1 * T2)};
    const int org[4] = {x[0] - l[0], x[1] - l[1], x[2] - l[2], x[3] - l[3]};
#pragma unroll
    for (int d = 0; d < 4; ++d) {
        nb[d][tid] = (x[d] + 1 == g.L[d]) ? s - (g.L[d] - 1) * g.stride_site[d] : s + g.stride_site[d];
        slots.zero(tid, d);
    }
    __syncthreads();
    T pl = T(0);
#pragma unroll 1
    for (int mu = 0; mu < 4; ++mu) {
        const T* __restrict__ umu_p = u.u[mu];
        const int tmu = mu == 0 ? T0 : (mu == 1 ? T1 : (mu == 2 ? T2 : T3));
        const int lsmu = mu == 0 ? 1 : (mu == 1 ? T0 : (mu == 2 ? T0 * T1 : T0 * T1 * T2));
        {  // (a) the thread's own three pairs
            const int xpmu = nb[mu][tid];
            const bool inside = coord_of(l, mu) + 1 < tmu;
            const Mat3<T> a = load_mat(umu_p, s);
            Mat3<T> acc = zero_mat<T>();
#pragma unroll 1
            for (int nu = 3; nu >= 0; --nu) {
                if (nu == mu) {
                    if (PLAQ && mu < 3) pl += re_tr_na(a, acc);  // acc = sum_{nu>mu} upper_{mu,nu}
                    continue;
                }
                const T* __restrict__ unu_p = u.u[nu];
                const Mat3<T> q = mul_nn(load_mat(unu_p, s), load_mat(umu_p, nb[nu][tid]));
                mac_na(acc, q, load_mat(unu_p, xpmu));
                if (inside) slots.add(tid + lsmu, nu, mul_an(a, q));
            }
            // (c) needs no barrier before it: slot[.][mu] has no other writer in this phase
            slots.add(tid, mu, acc);
        }
        {  // (b) lower staples entering through the low-mu face
            const int nface = NT / tmu;
#pragma unroll 1
            for (int i = tid; i < 3 * nface; i += NT) {
                const int k = i / nface;
                int j = i - k * nface;
                const int nu = k + (k >= mu ? 1 : 0);
                int lc[4];
                lc[0] = mu == 0 ? 0 : j % T0;
                if (mu != 0) j /= T0;
                lc[1] = mu == 1 ? 0 : j % T1;
                if (mu != 1) j /= T1;
                lc[2] = mu == 2 ? 0 : j % T2;
                if (mu != 2) j /= T2;
                lc[3] = mu == 3 ? 0 : j;
                const int li = lc[0] + T0 * (lc[1] + T1 * (lc[2] + T2 * lc[3]));
                const int gx[4] = {org[0] + lc[0], org[1] + lc[1], org[2] + lc[2], org[3] + lc[3]};
                const int sx = gx[0] + g.L[0] * (gx[1] + g.L[1] * (gx[2] + g.L[2] * gx[3]));
                const int sy = coord_of(gx, mu) == 0 ? sx + (g.L[mu] - 1) * g.stride_site[mu] : sx - g.stride_site[mu];
                const int syn = coord_of(gx, nu) + 1 == g.L[nu] ? sy - (g.L[nu] - 1) * g.stride_site[nu] : sy + g.stride_site[nu];
                const T* __restrict__ unu_p = u.u[nu];
                const Mat3<T> t = mul_an(load_mat(umu_p, sy), load_mat(unu_p, sy));
                slots.add(li, nu, mul_nn(t, load_mat(umu_p, syn)));
            }
        }
        __syncthreads();
    }
#pragma unroll 1
    for (int mu = 0; mu < 4; ++mu) store_mat(out.u[mu], s, smear_update(c0, c1, load_mat(u.u[mu], s), slots.get(tid, mu)));
    if (PLAQ) {
        double p[1] = {(double)pl};
        block_reduce_partial<1>(p, partials);
    }
}

template <typename T, typename MAP, int MINB>
int smear_shared_launch(lqx_ctx* ctx, const Links<T>& in, const LinksOut<T>& o, T c0, T c1, double* plaq) {
    const Geo& g = ctx->geo;
    const int grid = MAP::grid(g);
    const TileMap tm = MAP::map(g, kSlabZ);
    const size_t smem = sizeof(T) * 4 * 18 * MAP::THREADS + sizeof(int) * 4 * MAP::THREADS;
    // function attributes are per device: set on every call (microseconds) rather than cached per process
    if (plaq) LQX_CUDA(ctx, cudaFuncSetAttribute(k_smear_shared<T, true, MAP, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    else LQX_CUDA(ctx, cudaFuncSetAttribute(k_smear_shared<T, false, MAP, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (plaq) {
        int rc = lqx_ensure_partials(ctx, (size_t)grid);
        if (rc) return rc;
    }
    {
        LqxTimed timed(ctx, LQX_K_SMEAR);
        if (plaq) k_smear_shared<T, true, MAP, MINB><<<grid, MAP::THREADS, smem, ctx->stream>>>(g, tm, in, o, c0, c1, ctx->d_partials);
        else k_smear_shared<T, false, MAP, MINB><<<grid, MAP::THREADS, smem, ctx->stream>>>(g, tm, in, o, c0, c1, nullptr);
    }
    LQX_LAUNCH_CHECK(ctx);
    return plaq ? lqx_sum_partials(ctx, grid, 1, plaq) : LQX_OK;
}

// variant 4: four threads per site -- thread (site, mu) evaluates the six staples of ONE link, so a
// CTA of 4*TILE threads works on a TILE-site tile whose operand footprint (the tile, its faces and
// edges: ~15 matrices per site) is small enough to stay in L1 while 16 warps per SM hide latency.
// The literal kernel with one thread per site keeps three such footprints per SM alive and thrashes
// L1 (38 % hits, L2 -> L1 traffic at the L2 bandwidth limit; profiles/r01b).
template <typename T, bool PLAQ, typename MAP, int MINB>
__global__ void __launch_bounds__(MAP::THREADS * 4, MINB) k_smear_mu4(const __grid_constant__ Geo g, const __grid_constant__ TileMap tm,
                                                                      const __grid_constant__ Links<T> u, const __grid_constant__ LinksOut<T> out,
                                                                      T c0, T c1, double* __restrict__ partials, unsigned int* ticket,
                                                                      double* __restrict__ red_out) {
    __shared__ int nb[8][MAP::THREADS];  // [0..3] x+d^, [4..7] x-d^
    int x[4], s;
    double p[1] = {0.0};
    const int tid = threadIdx.x, mu = threadIdx.y;
    const bool valid = MAP::site(g, tm, x, s);
    if (valid && mu == 0) {
#pragma unroll
        for (int d = 0; d < 4; ++d) {
            nb[d][tid] = (x[d] + 1 == g.L[d]) ? s - (g.L[d] - 1) * g.stride_site[d] : s + g.stride_site[d];
            nb[4 + d][tid] = (x[d] == 0) ? s + (g.L[d] - 1) * g.stride_site[d] : s - g.stride_site[d];
        }
    }
    __syncthreads();
    if (valid) {
        T pl = T(0);
        const T* __restrict__ umu_p = u.u[mu];
        const int xpmu = nb[mu][tid];
        Mat3<T> acc = zero_mat<T>();
#pragma unroll 1
        for (int nu = 0; nu < 4; ++nu) {
            if (nu == mu) continue;
            const T* __restrict__ unu_p = u.u[nu];
            const int xpnu = nb[nu][tid], xmnu = nb[4 + nu][tid];
            {
                const Mat3<T> t = mul_nn(load_mat(unu_p, s), load_mat(umu_p, xpnu));
                if (PLAQ && mu < nu) {
                    const Mat3<T> up = mul_na(t, load_mat(unu_p, xpmu));
                    pl += re_tr_na(load_mat(umu_p, s), up);
                    add_to(acc, up);
                } else {
                    mac_na(acc, t, load_mat(unu_p, xpmu));
                }
            }
            {
                const Mat3<T> t = mul_an(load_mat(unu_p, xmnu), load_mat(umu_p, xmnu));
                mac_nn(acc, t, load_mat(unu_p, xmnu + (xpmu - s)));
            }
        }
        store_mat(out.u[mu], s, smear_update(c0, c1, load_mat(umu_p, s), acc));
        p[0] = (double)pl;
    }
    if (PLAQ) block_reduce_partial<1>(p, partials);
}

// tiles of the four-threads-per-site kernel: 64 sites (256 threads, two or three CTAs per SM) or
// 128 sites (512 threads, one CTA per SM)
typedef Tiled<8, 2, 2, 2> Tile64A;
typedef Tiled<16, 2, 2, 1> Tile64B;
typedef Tiled<4, 4, 2, 2> Tile64C;

template <typename T, typename MAP, int MINB>
int smear_mu4_launch(lqx_ctx* ctx, const Links<T>& in, const LinksOut<T>& o, T c0, T c1, double* plaq) {
    const Geo& g = ctx->geo;
    const int grid = MAP::grid(g);
    const TileMap tm = MAP::map(g, kSlabZ);
    if (plaq) {
        int rc = lqx_ensure_partials(ctx, (size_t)grid);
        if (rc) return rc;
    }
    const dim3 blk(MAP::THREADS, 4);
    LqxTimed timed(ctx, LQX_K_SMEAR);
    if (plaq) k_smear_mu4<T, true, MAP, MINB><<<grid, blk, 0, ctx->stream>>>(g, tm, in, o, c0, c1, ctx->d_partials, ctx->d_ticket, plaq);
    else k_smear_mu4<T, false, MAP, MINB><<<grid, blk, 0, ctx->stream>>>(g, tm, in, o, c0, c1, nullptr, nullptr, nullptr);
    LQX_LAUNCH_CHECK(ctx);
    return plaq ? lqx_sum_partials(ctx, grid, 1, plaq) : LQX_OK;
}

template <typename T>
int smear_launch_t(lqx_ctx* ctx, lqx_field* const uout[4], const lqx_field* const uin[4], double alpha, int only_mu,
                   double* plaq) {
    const Geo& g = ctx->geo;
    LinksOut<T> o;
    for (int mu = 0; mu < 4; ++mu) o.u[mu] = uout[mu] ? (T*)uout[mu]->data : nullptr;
    const Links<T> in = make_links<T>(uin);
    const T c0 = (T)(1.0 - alpha), c1 = (T)(alpha / 6.0);
    constexpr int PI = sizeof(T) == 4 ? 0 : 1;
    int variant = ctx->opt_smear_variant;
    const int tile_saved = ctx->opt_tile;
    if (variant == 0 && ctx->tuned_smear_variant[PI]) {  // the auto-tuner's choice, tile included
        variant = ctx->tuned_smear_variant[PI];
        if (ctx->opt_tile < 0) ctx->opt_tile = ctx->tuned_smear_tile[PI];
    }
    if (variant == 0) variant = lqx_smear_default_variant(ctx, sizeof(T) == 4 ? LQX_F32 : LQX_F64);
    struct Restore {
        lqx_ctx* c;
        int t;
        ~Restore() { c->opt_tile = t; }
    } restore = {ctx, tile_saved};
    // executed FMA lane-ops per site: 48 (variant 8: 42; variant 2: 36 + halo) products x 108 + update 4 x 36
    ctx->last_smear_lane_ops = 48 * 108 + 144;
    if (variant != 1 && variant != 2 && variant != 4 && variant != 6 && variant != 7 && variant != 8 && variant != 9 && variant != 10) variant = 3;
    if (only_mu >= 0) variant = 1;
    ctx->last_smear_variant = variant;
    ctx->last_smear_kernel = variant == 10 ? "k_smear_rowz" : variant == 9 ? "k_smear_rowlit" : variant == 8 ? "k_smear_rows" : variant == 7 ? "k_smear_tile"
                           : variant == 6 ? "k_smear_staged" : variant == 4 ? "k_smear_mu4" : variant == 2 ? "k_smear_shared"
                           : variant == 1 ? "k_smear_gather" : "k_smear_rolled";
    if (variant == 8 || variant == 10) ctx->last_smear_lane_ops = 42 * 108 + 144;
    if (variant == 2) ctx->last_smear_lane_ops = 36 * 108 + 144;  // + the halo products of the tile in use
    struct Fallback {  // a variant whose tiles do not fit hands over to the rolled kernel
        lqx_ctx* c;
        void operator()() const { c->last_smear_variant = 3, c->last_smear_kernel = "k_smear_rolled", c->last_smear_lane_ops = 48 * 108 + 144; }
    } fell_back = {ctx};
    if (variant == 10) {
        int rc = 1;
        if (sizeof(T) == 4) rc = lqx_smear_rowz_launch(ctx, reinterpret_cast<const Links<float>&>(in), reinterpret_cast<const LinksOut<float>&>(o), (float)c0, (float)c1, plaq);
        if (rc <= 0) return rc;
        variant = 9;  // fp64, or the lattice does not fit the eight-row tiles
        ctx->last_smear_variant = 9, ctx->last_smear_kernel = "k_smear_rowlit", ctx->last_smear_lane_ops = 48 * 108 + 144;
    }
    if (variant == 9) {
        const int rc = lqx_smear_rowlit_launch(ctx, in, o, c0, c1, plaq);
        if (rc <= 0) return rc;
        variant = 3;
        fell_back();
    }
    if (variant == 8) {
        int rc = 1;
        if (sizeof(T) == 4) rc = lqx_smear_rows_launch(ctx, reinterpret_cast<const Links<float>&>(in), reinterpret_cast<const LinksOut<float>&>(o), (float)c0, (float)c1, plaq);
        if (rc <= 0) return rc;
        variant = 3;  // fp64, or the lattice does not fit the row tiles
        fell_back();
    }
    if (variant == 7) {
        const int rc = lqx_smear_tile_launch(ctx, in, o, c0, c1, plaq);
        if (rc <= 0) return rc;
        variant = 3;  // no tile of this kernel divides the lattice
        fell_back();
    }
    if (variant == 6) {
        int rc = 1;
        if (sizeof(T) == 4) rc = lqx_smear_staged_launch(ctx, reinterpret_cast<const Links<float>&>(in), reinterpret_cast<const LinksOut<float>&>(o), (float)c0, (float)c1, plaq);
        if (rc <= 0) return rc;
        variant = 3;  // fp64, or the lattice is not a multiple of the staged kernel's tile
        fell_back();
    }
    if (variant == 2) {
        // option "tile": 1 = 8x4x4x2 (256 threads), 2 = 8x4x2x2, 3 = 4x4x4x2, 4 = 16x4x2x2 (256), 5 = 16x2x2x2
        const int t = ctx->opt_tile;
        int rc = 1;
        constexpr int MB256 = sizeof(T) == 4 ? 2 : 1, MB128 = sizeof(T) == 4 ? 4 : 2;
        if (sizeof(T) == 4 && (t == 1 || t < 0) && TileA::fits(g)) rc = smear_shared_launch<T, TileA, MB256>(ctx, in, o, c0, c1, plaq);
        else if (sizeof(T) == 4 && t == 4 && TileD::fits(g)) rc = smear_shared_launch<T, TileD, MB256>(ctx, in, o, c0, c1, plaq);
        else if ((t == 2 || t < 0) && TileB::fits(g)) rc = smear_shared_launch<T, TileB, MB128>(ctx, in, o, c0, c1, plaq);
        else if (t == 5 && TileE::fits(g)) rc = smear_shared_launch<T, TileE, MB128>(ctx, in, o, c0, c1, plaq);
        else if ((t == 3 || t < 0) && TileC::fits(g)) rc = smear_shared_launch<T, TileC, MB128>(ctx, in, o, c0, c1, plaq);
        if (rc <= 0) return rc;
        variant = 3;  // no tile of this kernel divides the lattice
        fell_back();
    }
    if (variant == 4) {
        // option "tile": 1 = 8x2x2x2, 2 = 16x2x2x1, 3 = 4x4x2x2 (64 sites); 4 = 8x4x2x2, 5 = 16x2x2x2 (128 sites)
        const int t = ctx->opt_tile;
        int rc = 1;
        constexpr int MB64 = sizeof(T) == 4 ? 3 : 1;
        if ((t == 1 || t < 0) && Tile64A::fits(g)) rc = smear_mu4_launch<T, Tile64A, MB64>(ctx, in, o, c0, c1, plaq);
        else if (t == 2 && Tile64B::fits(g)) rc = smear_mu4_launch<T, Tile64B, MB64>(ctx, in, o, c0, c1, plaq);
        else if ((t == 3 || t < 0) && Tile64C::fits(g)) rc = smear_mu4_launch<T, Tile64C, MB64>(ctx, in, o, c0, c1, plaq);
        else if (t == 4 && TileB::fits(g)) rc = smear_mu4_launch<T, TileB, 1>(ctx, in, o, c0, c1, plaq);
        else if (t == 5 && TileE::fits(g)) rc = smear_mu4_launch<T, TileE, 1>(ctx, in, o, c0, c1, plaq);
        if (rc <= 0) return rc;
        variant = 3;  // no tile of this kernel divides the lattice
        fell_back();
    }
    const int choice = lqx_pick_tile(ctx, sizeof(T) == 4 ? 1 : 0);  // measured best
    int nblocks = 0;
    LQX_WITH_MAP(choice, {
        const int grid = MAP::grid(g);
        nblocks = grid;
        const TileMap tm = MAP::map(g, kSlabZ);
        if (plaq) {
            int rc = lqx_ensure_partials(ctx, (size_t)grid);
            if (rc) return rc;
        }
        double* part = plaq ? ctx->d_partials : nullptr;
        unsigned int* tick = plaq ? ctx->d_ticket : nullptr;
        LqxTimed timed(ctx, LQX_K_SMEAR);
        if (variant == 1) {
            if (plaq) k_smear_gather<T, true, MAP><<<grid, MAP::THREADS, 0, ctx->stream>>>(g, tm, in, o, c0, c1, only_mu, part, tick, plaq);
            else k_smear_gather<T, false, MAP><<<grid, MAP::THREADS, 0, ctx->stream>>>(g, tm, in, o, c0, c1, only_mu, part, tick, plaq);
        } else {
            constexpr int MB = sizeof(T) == 4 ? (MAP::THREADS >= 256 ? 3 : 6) : (MAP::THREADS >= 256 ? 1 : 3);
            if (plaq) k_smear_rolled<T, true, MAP, MB><<<grid, MAP::THREADS, 0, ctx->stream>>>(g, tm, in, o, c0, c1, part, tick, plaq);
            else k_smear_rolled<T, false, MAP, MB><<<grid, MAP::THREADS, 0, ctx->stream>>>(g, tm, in, o, c0, c1, part, tick, plaq);
        }
    })
    LQX_LAUNCH_CHECK(ctx);
    return plaq ? lqx_sum_partials(ctx, nblocks, 1, plaq) : LQX_OK;
}

// one smear step restricted to the time slices [t0, t1): the rolled kernel on a sub-grid (streamed host path)
template <typename T>
int smear_range_t(lqx_ctx* ctx, lqx_field* const uout[4], const lqx_field* const uin[4], double alpha, int t0, int t1,
                  bool force_linear) {
    const Geo& g = ctx->geo;
    LinksOut<T> o;
    for (int mu = 0; mu < 4; ++mu) o.u[mu] = (T*)uout[mu]->data;
    const Links<T> in = make_links<T>(uin);
    const T c0 = (T)(1.0 - alpha), c1 = (T)(alpha / 6.0);
    const int choice = force_linear ? 0 : lqx_pick_tile(ctx, sizeof(T) == 4 ? 1 : 0);
    LQX_WITH_MAP(choice, {
        if (!MAP::splits_t(t0) || !MAP::splits_t(t1)) return 1;
        TileMap tm = MAP::map(g, kSlabZ);
        const int grid = MAP::restrict_t(g, tm, t0, t1);
        constexpr int MB = sizeof(T) == 4 ? (MAP::THREADS >= 256 ? 3 : 6) : (MAP::THREADS >= 256 ? 1 : 3);
        LqxTimed timed(ctx, LQX_K_SMEAR);
        k_smear_rolled<T, false, MAP, MB><<<grid, MAP::THREADS, 0, ctx->stream>>>(g, tm, in, o, c0, c1, nullptr, nullptr, nullptr);
    })
    LQX_LAUNCH_CHECK(ctx);
    return LQX_OK;
}

}  // namespace

int lqx_smear_default_variant(const lqx_ctx* ctx, lqx_prec prec) {
    const int pi = prec == LQX_F32 ? 0 : 1;
    if (ctx->opt_smear_variant) return ctx->opt_smear_variant;
    if (ctx->tuned_smear_variant[pi]) return ctx->tuned_smear_variant[pi];
    if (prec == LQX_F32 && lqx_smear_rowz_fits(ctx) && ctx->geo.L[0] * 8 > 256) return 10;
    return 9;
}

int lqx_smear_launch_range(lqx_ctx* ctx, lqx_field* const uout[4], const lqx_field* const uin[4], double alpha, int t0,
                           int t1) {
    // fp32: the kernel the whole-lattice step would run, on the range
    const int v32 = lqx_smear_default_variant(ctx, LQX_F32);
    if (uin[0]->prec == LQX_F32 && v32 == 10 && lqx_smear_rowz_fits(ctx)) {
        LinksOut<float> o;
        for (int mu = 0; mu < 4; ++mu) o.u[mu] = (float*)uout[mu]->data;
        return lqx_smear_rowz_launch_range(ctx, make_links<float>(uin), o, (float)(1.0 - alpha), (float)(alpha / 6.0), t0, t1);
    }
    if (uin[0]->prec == LQX_F32 && (v32 == 9 || v32 == 10)) {
        LinksOut<float> o;
        for (int mu = 0; mu < 4; ++mu) o.u[mu] = (float*)uout[mu]->data;
        const int rc9 = lqx_smear_rowlit_launch_range(ctx, make_links<float>(uin), o, (float)(1.0 - alpha), (float)(alpha / 6.0), t0, t1);
        if (rc9 != 1) return rc9;
    }
    int rc = uin[0]->prec == LQX_F32 ? smear_range_t<float>(ctx, uout, uin, alpha, t0, t1, false)
                                     : smear_range_t<double>(ctx, uout, uin, alpha, t0, t1, false);
    return rc;
}
// the same for ANY t0 < t1: where the 4-d tile in use does not split there, linear 128-site blocks do (every
// kernel map evaluates the same per-site arithmetic, so the output does not depend on the choice)
int lqx_smear_launch_range_any(lqx_ctx* ctx, lqx_field* const uout[4], const lqx_field* const uin[4], double alpha, int t0,
                               int t1) {
    int rc = lqx_smear_launch_range(ctx, uout, uin, alpha, t0, t1);
    if (rc != 1) return rc;
    return uin[0]->prec == LQX_F32 ? smear_range_t<float>(ctx, uout, uin, alpha, t0, t1, true)
                                   : smear_range_t<double>(ctx, uout, uin, alpha, t0, t1, true);
}

int lqx_smear_launch(lqx_ctx* ctx, lqx_field* const uout[4], const lqx_field* const uin[4], double alpha, int only_mu,
                     double* plaq) {
    return uin[0]->prec == LQX_F32 ? smear_launch_t<float>(ctx, uout, uin, alpha, only_mu, plaq)
                                   : smear_launch_t<double>(ctx, uout, uin, alpha, only_mu, plaq);
}
