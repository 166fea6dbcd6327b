// lqx staple sum + smear step with the CTA tile's own links held in shared memory
// (option "smear_variant" = 7, formula of BASELINE.json configs[0]).
//
// Why: profiles/r01j shows the rolled literal kernel moving 38.9 GB per launch from L2 into the SMs
// (lts__t_sectors_srcunit_tex_op_read x 32 B) in 3.26 ms = 11.9 TB/s, which is what the L2 -> SM fabric
// of this part delivers: three resident 256-site CTAs touch ~700 KB of operands per SM and L1 keeps 37 %.
// Three quarters of the 76 operand matrices a site reads belong to sites of its own tile.  Here every
// thread first copies the four links of ITS site into shared memory (same blocked layout as a field,
// the tile-local site index playing the role of the site index), and every operand whose site lies
// inside the tile is read from there; only the tile's halo goes to L1 / L2.  The choice is a select
// between two base pointers and two indices followed by ordinary (generic) loads, so a warp whose lanes
// straddle the tile edge does not diverge.  Same evaluation and summation order as k_smear_rolled:
// the two kernels agree bit for bit.
#include "lqx_smear.cuh"

namespace {

// all 18 reals of the colour matrix with index `idx` of a blocked array at `base` (shared or global)
template <typename T>
__device__ __forceinline__ Mat3<T> load_mat_generic(const T* base, int idx) {
    typedef typename Vec128<T>::type V;
    constexpr int W = Vec128<T>::W, NFULL = 18 / W;
    const T* blk = base + (size_t)(idx >> 5) * (32 * 18);
    const int lane = idx & 31;
    const V* p = reinterpret_cast<const V*>(blk) + lane;
    T r[18];
#pragma unroll
    for (int q = 0; q < NFULL; ++q) unpack(p[q * 32], &r[q * W]);
    if (18 % W != 0) {
        const float2 t = reinterpret_cast<const float2*>(blk + NFULL * 32 * W)[lane];
        r[NFULL * W] = (T)t.x;
        r[NFULL * W + 1] = (T)t.y;
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

template <typename T>
__device__ __forceinline__ Mat3<T> smear_update_t(T c0, T c1, const Mat3<T>& umu, const Mat3<T>& acc) {
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

template <typename T, bool PLAQ, typename MAP, int MINB>
__global__ void __launch_bounds__(MAP::THREADS, MINB) k_smear_tile(const __grid_constant__ Geo g, const __grid_constant__ TileMap tm,
                                                                   const __grid_constant__ Links<T> u, const __grid_constant__ LinksOut<T> out,
                                                                   T c0, T c1, double* __restrict__ partials) {
    constexpr int NT = MAP::THREADS;
    constexpr int LINK = 18 * NT;  // reals per link of the tile
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* tile = reinterpret_cast<T*>(smem_raw);                                 // [4][NT/32][18*32]
    int(*nb)[NT] = reinterpret_cast<int(*)[NT]>(smem_raw + sizeof(T) * 4 * LINK);  // [0..3] x+d^, [4..7] x-d^ (global site index)
    int x[4], s;
    MAP::site(g, tm, x, s);  // tiles always cover whole sites
    const int tid = threadIdx.x;
    const int l[4] = {tid % MAP::T0, (tid / MAP::T0) % MAP::T1, (tid / (MAP::T0 * MAP::T1)) % MAP::T2, tid / (MAP::T0 * MAP::T1 * MAP::T2)};
    constexpr int TD[4] = {MAP::T0, MAP::T1, MAP::T2, MAP::T3};
    constexpr int LS[4] = {1, MAP::T0, MAP::T0 * MAP::T1, MAP::T0 * MAP::T1 * MAP::T2};
    // bit d: x+d^ is a site of this tile; bit 4+d: x-d^ is
    unsigned inside = 0;
#pragma unroll
    for (int d = 0; d < 4; ++d) {
        nb[d][tid] = (x[d] + 1 == g.L[d]) ? s - (g.L[d] - 1) * g.stride_site[d] : s + g.stride_site[d];
        nb[4 + d][tid] = (x[d] == 0) ? s + (g.L[d] - 1) * g.stride_site[d] : s - g.stride_site[d];
        if (l[d] + 1 < TD[d]) inside |= 1u << d;
        if (l[d] > 0) inside |= 1u << (4 + d);
    }
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        T r[18];
        load_site<T, 18>(u.u[mu], s, r);
        store_site<T, 18>(tile + mu * LINK, tid, r);
    }
    __syncthreads();

    double p[1] = {0.0};
    T pl = T(0);
#pragma unroll 1
    for (int mu = 0; mu < 4; ++mu) {
        const T* umu_g = u.u[mu];
        const T* umu_t = tile + mu * LINK;
        const int xpmu = nb[mu][tid];
        const bool in_pmu = (inside >> mu) & 1u;
        const int ls_mu = mu == 0 ? LS[0] : (mu == 1 ? LS[1] : (mu == 2 ? LS[2] : LS[3]));
        Mat3<T> acc = zero_mat<T>();
#pragma unroll 1
        for (int nu = 3; nu >= 0; --nu) {  // upper: U_nu(x) U_mu(x+nu^) adj(U_nu(x+mu^))
            if (nu == mu) continue;
            const T* unu_g = u.u[nu];
            const T* unu_t = tile + nu * LINK;
            const int ls_nu = nu == 0 ? LS[0] : (nu == 1 ? LS[1] : (nu == 2 ? LS[2] : LS[3]));
            const bool in_pnu = (inside >> nu) & 1u;
            const Mat3<T> t = mul_nn(load_mat_generic(unu_t, tid),
                                     load_mat_generic(in_pnu ? umu_t : umu_g, in_pnu ? tid + ls_nu : nb[nu][tid]));
            mac_na(acc, t, load_mat_generic(in_pmu ? unu_t : unu_g, in_pmu ? tid + ls_mu : xpmu));
        }
#pragma unroll 1
        for (int nu = 0; nu < 4; ++nu) {  // lower: adj(U_nu(x-nu^)) U_mu(x-nu^) U_nu(x-nu^+mu^)
            if (nu == mu) continue;
            const T* unu_g = u.u[nu];
            const T* unu_t = tile + nu * LINK;
            const int ls_nu = nu == 0 ? LS[0] : (nu == 1 ? LS[1] : (nu == 2 ? LS[2] : LS[3]));
            const bool in_mnu = (inside >> (4 + nu)) & 1u;
            const int xmnu = nb[4 + nu][tid];
            const int i1 = in_mnu ? tid - ls_nu : xmnu;
            const Mat3<T> t = mul_an(load_mat_generic(in_mnu ? unu_t : unu_g, i1), load_mat_generic(in_mnu ? umu_t : umu_g, i1));
            const bool in_d = in_mnu && in_pmu;
            mac_nn(acc, t, load_mat_generic(in_d ? unu_t : unu_g, in_d ? tid - ls_nu + ls_mu : xmnu + (xpmu - s)));
        }
        const Mat3<T> umu = load_mat_generic(umu_t, tid);
        if (PLAQ) pl += re_tr_na(umu, acc);
        store_mat(out.u[mu], s, smear_update_t(c0, c1, umu, acc));
    }
    p[0] = 0.25 * (double)pl;
    if (PLAQ) block_reduce_partial<1>(p, partials);
}

template <typename T, typename MAP, int MINB>
int tile_launch(lqx_ctx* ctx, const Links<T>& in, const LinksOut<T>& o, T c0, T c1, double* plaq) {
    const Geo& g = ctx->geo;
    const int grid = MAP::grid(g);
    const TileMap tm = MAP::map(g, kSlabZ);
    const size_t smem = sizeof(T) * 4 * 18 * MAP::THREADS + sizeof(int) * 8 * MAP::THREADS;
    if (plaq) LQX_CUDA(ctx, cudaFuncSetAttribute(k_smear_tile<T, true, MAP, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    else LQX_CUDA(ctx, cudaFuncSetAttribute(k_smear_tile<T, false, MAP, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (plaq) {
        int rc = lqx_ensure_partials(ctx, (size_t)grid);
        if (rc) return rc;
    }
    {
        LqxTimed timed(ctx, LQX_K_SMEAR);
        if (plaq) k_smear_tile<T, true, MAP, MINB><<<grid, MAP::THREADS, smem, ctx->stream>>>(g, tm, in, o, c0, c1, ctx->d_partials);
        else k_smear_tile<T, false, MAP, MINB><<<grid, MAP::THREADS, smem, ctx->stream>>>(g, tm, in, o, c0, c1, nullptr);
    }
    LQX_LAUNCH_CHECK(ctx);
    return plaq ? lqx_sum_partials(ctx, grid, 1, plaq) : LQX_OK;
}

template <typename T>
int tile_dispatch(lqx_ctx* ctx, const Links<T>& in, const LinksOut<T>& o, T c0, T c1, double* plaq) {
    const Geo& g = ctx->geo;
    const int t = ctx->opt_tile;  // 1 = 8x4x4x2 (256 threads), 2 = 8x4x2x2, 3 = 4x4x4x2, 4 = 16x4x2x2 (256), 5 = 16x2x2x2
    constexpr bool F = sizeof(T) == 4;
    // fp32: 256-site tiles are 80 KB of shared memory (two CTAs per SM), 128-site tiles 40 KB (four);
    // fp64: 128-site tiles are 78 KB (two CTAs per SM)
    if (F && (t == 1 || t < 0) && TileA::fits(g)) return tile_launch<T, TileA, 2>(ctx, in, o, c0, c1, plaq);
    if (F && t == 4 && TileD::fits(g)) return tile_launch<T, TileD, 2>(ctx, in, o, c0, c1, plaq);
    if ((t == 2 || t < 0) && TileB::fits(g)) return tile_launch<T, TileB, F ? 4 : 2>(ctx, in, o, c0, c1, plaq);
    if (t == 5 && TileE::fits(g)) return tile_launch<T, TileE, F ? 4 : 2>(ctx, in, o, c0, c1, plaq);
    if ((t == 3 || t < 0) && TileC::fits(g)) return tile_launch<T, TileC, F ? 4 : 2>(ctx, in, o, c0, c1, plaq);
    return 1;
}

}  // namespace

int lqx_smear_tile_launch(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, double* plaq) {
    return tile_dispatch<float>(ctx, in, out, c0, c1, plaq);
}
int lqx_smear_tile_launch(lqx_ctx* ctx, const Links<double>& in, const LinksOut<double>& out, double c0, double c1, double* plaq) {
    return tile_dispatch<double>(ctx, in, out, c0, c1, plaq);
}
