// lqx staple sum + smear step, fp32, plane-ordered evaluation on whole-x-row tiles held in shared memory
// (option "smear_variant" = 8, formula of BASELINE.json configs[0]).
//
// What bounds the literal kernel (profiles/r02b): 76 operand matrices per site through the 128 B/clk L1
// data pipe (1986 wavefronts per warp, pipe 75 % busy: x-shifted rows of an 8-site-wide tile straddle two
// lines, +24 %) and 39 GB per launch from L2 (12.7 TB/s, the fabric's limit).  This kernel attacks both:
//
//  * evaluation order: the six planes (mu < nu) one after the other with all four staple sums S_mu live.
//    With B = U_nu(x+mu^), C = U_mu(x+nu^) the product Z = B adj(C) serves BOTH upper staples of the plane,
//    S_nu += U_mu(x) Z and S_mu += U_nu(x) adj(Z): 3 products instead of 4, and 42 products / 64 operand
//    fetches per site instead of 48 / 76.  (Algebra of DESIGN.md sec.6.1; the oracle stays literal.)
//  * tile = ROWS whole x-rows (L0 x 2 x 2 x 2 sites, one thread per site), the tile's own links copied to
//    shared memory in the blocked field layout.  x-neighbours wrap around inside the row, so they are
//    ALWAYS in the tile and come out of shared memory at any alignment for 4 wavefronts per 128-bit chunk;
//    y/z/t-neighbours are in the tile for half of the rows.  Each operand is fetched by generic loads from a
//    SELECTED address (tile in shared memory or field in global memory): nothing diverges, and a warp mixes the
//    two spaces only where it straddles two rows of different y/z/t position (see fetch_mat).
//  * persistent CTAs, one per SM, double-buffered: while tile k is multiplied the own links of tile k+1
//    arrive by cp.async, so the fill never idles the FMA pipe and one barrier per tile suffices.
//  * option "tile" = 6 / 7: one 2x2x1-row tile per CTA and one buffer, two CTAs per SM, so that the SM keeps an L1;
//    7 requests every halo operand with prefetch.global.L1 three products ahead of its load (pf_mat).  Measured at
//    48^3x96: persistent form 4.8 ms, 6: 3.76 ms, 7: 2.84 ms -- level with the literal row-tile kernel (variant 9,
//    2.83 ms) at half its warps (profiles/r02j).
//
// Sums the staples of a link in plane order (not the oracle's nu-ascending order): agrees with the other
// variants to rounding, not bit for bit.
#include <cuda_pipeline.h>

#include "lqx_smear.cuh"

namespace {

struct RowMap {
    int ny, nz, nt;  // tiles per direction
    int zs;          // z-tiles per slab: tiles are visited y, z fastest inside a slab, then t, then the next slab,
                     // so that the +-t neighbour rows of a tile are still in L2 (as Tiled<>::site does)
    int ntiles;
    int toff;        // first t-tile of the launch (a launch may cover a range of time slices: streamed host path, t-split)
};

// One colour matrix from the tile in shared memory (in) or from the field in global memory, by GENERIC loads from a
// selected address.  Two facts shape this: (1) a predicated pair ld.shared / ld.global into the same registers --
// written by hand or produced by ptxas if-converting a branch -- never ends a live range, and ptxas then keeps the
// destination registers of all 64 fetches alive at once (5.5 KB of spills per thread); (2) x-neighbours are always in
// the tile, so a warp mixes the two spaces only where it straddles two rows with different y/z/t position.
// Cache operator: .cg (SASS LD.E.128.STRONG.GPU) -- the halo is served by L2, the few KB of L1 beside two 108 KB tiles
// hit 4 % of the time; measured 0.5-1.0 % faster than the default at 48^3x96 (2.866 -> 2.851 ms on eight-row tiles,
// 2.845 -> 2.816 on four-row tiles); L1::no_allocate and L1::evict_first are 20-50 % SLOWER (3.48-4.24 ms), the
// L2::128B / L2::256B prefetch-size hints change nothing.  Lanes that address the tile in shared memory ignore it.
__device__ __forceinline__ Mat3<float> fetch_mat(unsigned long long s_link, const float* g_link, bool in, int li, int gi) {
    const int idx = in ? li : gi;
    const unsigned off = (unsigned)(idx >> 5) * (32u * 18u * 4u) + (unsigned)(idx & 31) * 16u;
    const unsigned long long a = (in ? s_link : (unsigned long long)g_link) + off;
    const unsigned half = 2048u - (unsigned)(idx & 31) * 8u;
    float r[18];
#pragma unroll
    for (int q = 0; q < 4; ++q)
        asm volatile("ld.cg.v4.f32 {%0,%1,%2,%3}, [%4];"
                     : "=f"(r[4 * q]), "=f"(r[4 * q + 1]), "=f"(r[4 * q + 2]), "=f"(r[4 * q + 3])
                     : "l"(a + q * 512u));
    asm volatile("ld.cg.v2.f32 {%0,%1}, [%2];" : "=f"(r[16]), "=f"(r[17]) : "l"(a + half));
    Mat3<float> m;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            m.re[i][j] = r[2 * (3 * i + j)];
            m.im[i][j] = r[2 * (3 * i + j) + 1];
        }
    return m;
}
// a matrix of the tile itself (always shared memory)
__device__ __forceinline__ Mat3<float> fetch_own(unsigned long long s_link_generic, int li) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(reinterpret_cast<const void*>(s_link_generic)) + (unsigned)(li >> 5) * (32u * 18u * 4u) + (unsigned)(li & 31) * 16u;
    const unsigned half = 2048u - (unsigned)(li & 31) * 8u;
    float r[18];
#pragma unroll
    for (int q = 0; q < 4; ++q)
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];"
                     : "=f"(r[4 * q]), "=f"(r[4 * q + 1]), "=f"(r[4 * q + 2]), "=f"(r[4 * q + 3])
                     : "r"(sa + q * 512u));
    asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(r[16]), "=f"(r[17]) : "r"(sa + half));
    Mat3<float> m;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            m.re[i][j] = r[2 * (3 * i + j)];
            m.im[i][j] = r[2 * (3 * i + j) + 1];
        }
    return m;
}

// the four links of site s -> shared buffer slot li, asynchronously (4 x 16 B + 8 B per link); the lines are marked
// evict-last in L2 (the neighbouring tiles read them again as their halo): 2.836 -> 2.830 ms, 2.805 -> 2.798 on four-row tiles
__device__ __forceinline__ void fill_async(float* buf, int link_floats, const Links<float>& u, int s, int li) {
    unsigned long long pol;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    const size_t goff = (size_t)(s >> 5) * (32 * 18) + (size_t)(s & 31) * 4;
    const int soff = (li >> 5) * (32 * 18) + (li & 31) * 4;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        const float* g = u.u[mu] + goff;
        float* d = buf + mu * link_floats + soff;
#pragma unroll
        for (int q = 0; q < 4; ++q)
            asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"((unsigned)__cvta_generic_to_shared(d + q * 128)), "l"(g + q * 128), "l"(pol) : "memory");
        asm volatile("cp.async.ca.shared.global.L2::cache_hint [%0], [%1], 8, %2;" ::"r"((unsigned)__cvta_generic_to_shared(d + 512 - (li & 31) * 2)), "l"(g + 512 - (s & 31) * 2), "l"(pol) : "memory");
    }
}

// fp64 forms of the three helpers (variant 9 in double precision): a matrix is nine 128-bit chunks of two doubles,
// 4608 bytes per 32-site block, no trailing half chunk
__device__ __forceinline__ Mat3<double> fetch_mat(unsigned long long s_link, const double* g_link, bool in, int li, int gi) {
    const int idx = in ? li : gi;
    const unsigned long long off = (unsigned long long)(idx >> 5) * (32u * 18u * 8u) + (unsigned)(idx & 31) * 16u;
    const unsigned long long a = (in ? s_link : (unsigned long long)g_link) + off;
    double r[18];
#pragma unroll
    for (int q = 0; q < 9; ++q) asm volatile("ld.cg.v2.f64 {%0,%1}, [%2];" : "=d"(r[2 * q]), "=d"(r[2 * q + 1]) : "l"(a + q * 512u));
    Mat3<double> m;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            m.re[i][j] = r[2 * (3 * i + j)];
            m.im[i][j] = r[2 * (3 * i + j) + 1];
        }
    return m;
}
__device__ __forceinline__ Mat3<double> fetch_own_d(unsigned long long s_link_generic, int li) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(reinterpret_cast<const void*>(s_link_generic)) + (unsigned)(li >> 5) * (32u * 18u * 8u) + (unsigned)(li & 31) * 16u;
    double r[18];
#pragma unroll
    for (int q = 0; q < 9; ++q) asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(r[2 * q]), "=d"(r[2 * q + 1]) : "r"(sa + q * 512u));
    Mat3<double> m;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            m.re[i][j] = r[2 * (3 * i + j)];
            m.im[i][j] = r[2 * (3 * i + j) + 1];
        }
    return m;
}
__device__ __forceinline__ void fill_async(double* buf, int link_reals, const Links<double>& u, int s, int li) {
    unsigned long long pol;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    const size_t goff = (size_t)(s >> 5) * (32 * 18) + (size_t)(s & 31) * 2;
    const int soff = (li >> 5) * (32 * 18) + (li & 31) * 2;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        const double* g = u.u[mu] + goff;
        double* d = buf + mu * link_reals + soff;
#pragma unroll
        for (int q = 0; q < 9; ++q)
            asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"((unsigned)__cvta_generic_to_shared(d + q * 64)), "l"(g + q * 64), "l"(pol) : "memory");
    }
}
template <typename T>
__device__ __forceinline__ Mat3<T> fetch_own_t(unsigned long long s_link_generic, int li);
template <>
__device__ __forceinline__ Mat3<float> fetch_own_t<float>(unsigned long long a, int li) { return fetch_own(a, li); }
template <>
__device__ __forceinline__ Mat3<double> fetch_own_t<double>(unsigned long long a, int li) { return fetch_own_d(a, li); }

// The tile's own links by TMA bulk copies (cp.async.bulk, SASS UBLKCP; option "bulk_fill" = 1): where the RY rows of one
// (z, t) position are a whole number of 32-site blocks, they are ONE contiguous byte range of a link field and of the tile
// buffer alike (the blocked layout is the same on both sides), so a tile is RZ*RT*4 copies issued by the lanes of one warp
// and awaited on an mbarrier -- instead of 20 LDGSTS per thread, whose 72 shared-memory write wavefronts per warp ride the
// L1 data pipe the staple sum is short of (4.5 % of the kernel's wavefronts) and whose 240 warp instructions per tile take
// issue slots.  Bit-identical output; MEASURED SLOWER at 48^3x96: 2.91 ms against 2.87 ms with sixteen 6912-byte copies
// per tile (four-row tiles: 2.87 against 2.85), 3.05 ms with forty-eight 2304-byte copies -- a tile's 110 KB arrive later through the copy engine than through
// 384 threads' LDGSTS, and while a CTA waits for its tile the SM runs on the other CTA's twelve warps alone.  Kept as an
// option and as the measurement; the default fill stays cp.async.
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    unsigned ok = 0;
    while (!ok)
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
}

// scheduling fence: every element of m must exist before any later (volatile) load is issued.  Without it the
// compiler hoists the independent operand loads of all six planes to the top and spills kilobytes per thread.
__device__ __forceinline__ void fence_mat(const Mat3<float>& m) {
    asm volatile("" ::"f"(m.re[0][0]), "f"(m.re[0][1]), "f"(m.re[0][2]), "f"(m.re[1][0]), "f"(m.re[1][1]), "f"(m.re[1][2]),
                 "f"(m.re[2][0]), "f"(m.re[2][1]), "f"(m.re[2][2]), "f"(m.im[0][0]), "f"(m.im[0][1]), "f"(m.im[0][2]),
                 "f"(m.im[1][0]), "f"(m.im[1][1]), "f"(m.im[1][2]), "f"(m.im[2][0]), "f"(m.im[2][1]), "f"(m.im[2][2]));
}


// What a thread knows about its site, packed so that it costs four registers and not twenty-four (the kernel runs
// at the 168-register limit of twelve warps per SM): everything else is re-derived per fetch from uniform values.
//   mask bit d      : x+d^ is in the tile          bit 4+d  : x-d^ is in the tile
//        bit 8+d    : x_d + 1 == L_d (x+d^ wraps)  bit 12+d : x_d == 0 (x-d^ wraps)
struct SiteCtx {
    int s;         // global site index
    unsigned mask;
    int dpx, dmx;  // tile-local index delta of x+0^ / x-0^ (the row wraps around inside the tile)
    int row_y, row_z, row_t;  // tile-local index delta of one step in y, z, t (uniform)
    template <int D>
    __device__ __forceinline__ bool ip() const { return D == 0 ? true : (mask >> D) & 1u; }
    template <int D>
    __device__ __forceinline__ bool im() const { return D == 0 ? true : (mask >> (4 + D)) & 1u; }
    template <int D>
    __device__ __forceinline__ int dp() const { return D == 0 ? dpx : (D == 1 ? row_y : (D == 2 ? row_z : row_t)); }
    template <int D>
    __device__ __forceinline__ int dm() const { return D == 0 ? dmx : -(D == 1 ? row_y : (D == 2 ? row_z : row_t)); }
    // global site index of x+d^ / x-d^
    template <int D>
    __device__ __forceinline__ int gp(const Geo& g) const {
        return ((mask >> (8 + D)) & 1u) ? s - (g.L[D] - 1) * g.stride_site[D] : s + g.stride_site[D];
    }
    template <int D>
    __device__ __forceinline__ int gm(const Geo& g) const {
        return ((mask >> (12 + D)) & 1u) ? s + (g.L[D] - 1) * g.stride_site[D] : s - g.stride_site[D];
    }
};

// the operands of one plane mu < nu, in the order they are consumed:
//   B = U_nu(x+mu), C = U_mu(x+nu)                      Z = B adj(C)
//   U_mu(x)                                             S_nu += U_mu(x) Z        upper staple of link nu
//   U_nu(x)                                             S_mu += U_nu(x) adj(Z)   upper staple of link mu
//   E = U_nu(x-nu), F = U_mu(x-nu), G = U_nu(x-nu+mu)   S_mu += (adj(E) F) G     lower staple of link mu
//   E' = U_mu(x-mu), F' = U_nu(x-mu), G' = U_mu(x-mu+nu) S_nu += (adj(E') F') G' lower staple of link nu
// The loads of every product are issued BEFORE the FMAs of the product in front of it (one product of
// prefetch); fence_mat pins that order.  B and C of the next plane are fetched during this plane's last product.
// L1 prefetch of a halo matrix (nothing for a matrix of the tile): five lines per warp and chunk, no destination
// register, so ptxas cannot sink it to a use -- the only way found to put a request AHEAD of the products at the
// register limit.  Needs an L1 to land in: used by the two-CTAs-per-SM form (one tile buffer each), not by the
// persistent double-buffered form whose shared memory takes the whole SM.
__device__ __forceinline__ void pf_mat(const float* g_link, bool in, int gi) {
    if (!in) {
        const char* a = reinterpret_cast<const char*>(g_link) + (size_t)(gi >> 5) * (32 * 18 * 4) + (size_t)(gi & 31) * 16;
#pragma unroll
        for (int q = 0; q < 4; ++q) asm volatile("prefetch.global.L1 [%0];" ::"l"(a + q * 512));
        asm volatile("prefetch.global.L1 [%0];" ::"l"(a + 2048 - (gi & 31) * 8));
    }
}

template <int MU, int NU>
__device__ __forceinline__ void fetch_BC(Mat3<float>& B, Mat3<float>& C, const SiteCtx& c, int li, const unsigned long long (&sl)[4],
                                         const Links<float>& u, const Geo& g) {
    B = fetch_mat(sl[NU], u.u[NU], c.ip<MU>(), li + c.dp<MU>(), c.gp<MU>(g));
    C = fetch_mat(sl[MU], u.u[MU], c.ip<NU>(), li + c.dp<NU>(), c.gp<NU>(g));
}

template <int MU, int NU, int MU2, int NU2, bool PF, bool FENCE>
__device__ __forceinline__ void plane(Mat3<float> (&S)[4], Mat3<float>& B, Mat3<float>& C, const SiteCtx& c, int li,
                                      const unsigned long long (&sl)[4], const Links<float>& u, const Geo& g) {
    constexpr int M2 = MU2 >= 0 ? MU2 : 0, N2 = NU2 >= 0 ? NU2 : 1;
    // PF: the halo operands are requested into L1 three products ahead of their loads, in three groups spread over the
    // plane (all at the plane's start measured slower: 2.99 against 2.84 ms).  With the requests under way the
    // scheduling fences below only cost (2.88 -> 2.84 ms without them), so the PF form leaves the order to ptxas.
    if (PF) {  // the first lower staple's E, F, G
        pf_mat(u.u[NU], c.im<NU>(), c.gm<NU>(g));
        pf_mat(u.u[MU], c.im<NU>(), c.gm<NU>(g));
        pf_mat(u.u[NU], c.im<NU>() && c.ip<MU>(), c.gm<NU>(g) + (c.gp<MU>(g) - c.s));
    }
    // Software pipeline, one product deep: the operand(s) of the next product are requested, then __syncwarp() --
    // a memory-ordering point ptxas will not sink loads across (left alone it moves every load down to its first
    // use to save registers, and twelve warps per SM cannot cover an L2 round trip per operand) -- then the FMAs of
    // the current product.  Four operand matrices live beside the four staple sums at the widest point.
    const Mat3<float> Amu = fetch_own(sl[MU], li);
    if (FENCE) __syncwarp();
    const Mat3<float> Z = mul_na(B, C);
    if (FENCE) fence_mat(Z);
    const Mat3<float> Anu = fetch_own(sl[NU], li);
    if (FENCE) __syncwarp();
    if (PF) {  // the second lower staple's E', F', G'
        pf_mat(u.u[MU], c.im<MU>(), c.gm<MU>(g));
        pf_mat(u.u[NU], c.im<MU>(), c.gm<MU>(g));
        pf_mat(u.u[MU], c.im<MU>() && c.ip<NU>(), c.gm<MU>(g) + (c.gp<NU>(g) - c.s));
    }
    mac_nn(S[NU], Amu, Z);
    if (FENCE) fence_mat(S[NU]);
    const Mat3<float> E = fetch_mat(sl[NU], u.u[NU], c.im<NU>(), li + c.dm<NU>(), c.gm<NU>(g));
    const Mat3<float> F = fetch_mat(sl[MU], u.u[MU], c.im<NU>(), li + c.dm<NU>(), c.gm<NU>(g));
    if (FENCE) __syncwarp();
    mac_na(S[MU], Anu, Z);
    if (FENCE) fence_mat(S[MU]);
    const Mat3<float> G = fetch_mat(sl[NU], u.u[NU], c.im<NU>() && c.ip<MU>(), li + c.dm<NU>() + c.dp<MU>(), c.gm<NU>(g) + (c.gp<MU>(g) - c.s));
    if (FENCE) __syncwarp();
    if (PF && MU2 >= 0) {  // the next plane's B and C
        pf_mat(u.u[N2], c.ip<M2>(), c.gp<M2>(g));
        pf_mat(u.u[M2], c.ip<N2>(), c.gp<N2>(g));
    }
    const Mat3<float> t = mul_an(E, F);
    if (FENCE) fence_mat(t);
    const Mat3<float> E2 = fetch_mat(sl[MU], u.u[MU], c.im<MU>(), li + c.dm<MU>(), c.gm<MU>(g));
    const Mat3<float> F2 = fetch_mat(sl[NU], u.u[NU], c.im<MU>(), li + c.dm<MU>(), c.gm<MU>(g));
    if (FENCE) __syncwarp();
    mac_nn(S[MU], t, G);
    if (FENCE) fence_mat(S[MU]);
    const Mat3<float> G2 = fetch_mat(sl[MU], u.u[MU], c.im<MU>() && c.ip<NU>(), li + c.dm<MU>() + c.dp<NU>(), c.gm<MU>(g) + (c.gp<NU>(g) - c.s));
    if (FENCE) __syncwarp();
    const Mat3<float> t2 = mul_an(E2, F2);
    if (FENCE) fence_mat(t2);
    if (MU2 >= 0) {
        B = fetch_mat(sl[N2], u.u[N2], c.ip<M2>(), li + c.dp<M2>(), c.gp<M2>(g));
        C = fetch_mat(sl[M2], u.u[M2], c.ip<N2>(), li + c.dp<N2>(), c.gp<N2>(g));
        if (FENCE) __syncwarp();
    }
    mac_nn(S[NU], t2, G2);
    if (FENCE) fence_mat(S[NU]);
}

template <bool PLAQ, int RY, int RZ, int RT, int MAXT, int MINB, bool PF>
__global__ void __launch_bounds__(MAXT, MINB) k_smear_rows(const __grid_constant__ Geo g, const __grid_constant__ RowMap rm,
                                                        const __grid_constant__ Links<float> u, const __grid_constant__ LinksOut<float> out,
                                                        float c0, float c1, double* __restrict__ partials) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int L0 = g.L[0];
    const int nthr = blockDim.x;  // L0 * RY * RZ * RT
    const int npad = (nthr + 31) & ~31;
    const int link_floats = 18 * npad;
    float* const buf0 = reinterpret_cast<float*>(smem_raw);
    const int li = threadIdx.x;
    const int lx = li % L0, row = li / L0;
    const int ly = row % RY, lz = (row / RY) % RZ, lt = row / (RY * RZ);

    SiteCtx c;
    // tile-local deltas and in-tile flags do not depend on the tile; x-neighbours wrap around inside the row
    c.dpx = (lx + 1 == L0) ? -(L0 - 1) : 1;
    c.dmx = (lx == 0) ? (L0 - 1) : -1;
    c.row_y = L0, c.row_z = RY * L0, c.row_t = RY * RZ * L0;
    const unsigned tile_mask = (ly + 1 < RY ? 2u : 0u) | (lz + 1 < RZ ? 4u : 0u) | (lt + 1 < RT ? 8u : 0u) | (ly > 0 ? 32u : 0u) |
                               (lz > 0 ? 64u : 0u) | (lt > 0 ? 128u : 0u);

    const int per_slab = rm.ny * rm.zs * rm.nt;
    auto site_of = [&](int tile, int (&x)[4]) {
        const int k = tile / per_slab;
        int rem = tile - k * per_slab;
        const int bt = rem / (rm.ny * rm.zs);
        rem -= bt * (rm.ny * rm.zs);
        const int bz = rem / rm.ny + k * rm.zs, by = rem % rm.ny;
        x[0] = lx, x[1] = RY * by + ly, x[2] = RZ * bz + lz, x[3] = RT * bt + lt;
        return x[0] + g.L[0] * (x[1] + g.L[1] * (x[2] + g.L[2] * x[3]));
    };

    float pl = 0.f;
    int tile = blockIdx.x;
    int cur = 0;
    if (tile < rm.ntiles) {
        int x[4];
        const int s = site_of(tile, x);
        fill_async(buf0, link_floats, u, s, li);
    }
    __pipeline_commit();
    for (; tile < rm.ntiles; tile += gridDim.x, cur ^= 1) {
        int x[4];
        c.s = site_of(tile, x);
        c.mask = tile_mask;
#pragma unroll
        for (int d = 0; d < 4; ++d) {
            if (x[d] + 1 == g.L[d]) c.mask |= 1u << (8 + d);
            if (x[d] == 0) c.mask |= 1u << (12 + d);
        }
        __pipeline_wait_prior(0);
        __syncthreads();  // buffer `cur` is complete, and every thread is done with buffer cur^1
        {
            const int next = tile + gridDim.x;
            if (next < rm.ntiles) {
                int xn[4];
                const int sn = site_of(next, xn);
                fill_async(buf0 + (cur ^ 1) * 4 * link_floats, link_floats, u, sn, li);
            }
            __pipeline_commit();
        }
        unsigned long long sl[4];  // generic addresses of the four links of the current buffer
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) sl[mu] = (unsigned long long)(buf0 + (cur * 4 + mu) * link_floats);

        Mat3<float> S[4];
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) S[mu] = zero_mat<float>();
        constexpr bool FENCE = !PF || PLAQ;
        Mat3<float> B, C;
        fetch_BC<0, 1>(B, C, c, li, sl, u, g);
        plane<0, 1, 0, 2, PF, FENCE>(S, B, C, c, li, sl, u, g);
        plane<0, 2, 0, 3, PF, FENCE>(S, B, C, c, li, sl, u, g);
        plane<0, 3, 1, 2, PF, FENCE>(S, B, C, c, li, sl, u, g);
        plane<1, 2, 1, 3, PF, FENCE>(S, B, C, c, li, sl, u, g);
        plane<1, 3, 2, 3, PF, FENCE>(S, B, C, c, li, sl, u, g);
        plane<2, 3, -1, -1, PF, FENCE>(S, B, C, c, li, sl, u, g);
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            const Mat3<float> umu = fetch_own(sl[mu], li);
            Mat3<float> r;
            float tr = 0.f;
#pragma unroll
            for (int i = 0; i < 3; ++i)
#pragma unroll
                for (int j = 0; j < 3; ++j) {  // trace and update element by element: r takes S's registers
                    if (PLAQ) tr = fmaf(umu.re[i][j], S[mu].re[i][j], tr);
                    if (PLAQ) tr = fmaf(umu.im[i][j], S[mu].im[i][j], tr);
                    r.re[i][j] = fmaf(c1, S[mu].re[i][j], c0 * umu.re[i][j]);
                    r.im[i][j] = fmaf(c1, S[mu].im[i][j], c0 * umu.im[i][j]);
                }
            if (PLAQ) pl += tr;
            store_mat(out.u[mu], c.s, r);
        }
    }
    __pipeline_wait_prior(0);
    if (PLAQ) {
        double p[1] = {0.25 * (double)pl};
        block_reduce_partial<1>(p, partials);
    }
}

// Tensor memory as a per-thread operand store (sm_100a).  TMEM is 512 columns x 128 lanes x 32 bit per SM with its own
// read / write pipes (LDTM 64 B/clk, STTM 256 B/clk per SM, B300_MICROARCH.md), beside the 128 B/clk L1 / shared data pipe
// the staple sum is short of; a warp reaches the 32 lanes of its quarter (warp id mod 4) and every thread its own lane, so
// it can hold exactly what a thread re-reads of its OWN site: the four links of the site (72 words), fetched 16 times per
// site update.  No tensor-core instruction is involved: tcgen05.alloc / st / ld / dealloc only.
// Measured (option "tile" = 7 of variant 9; output bit-identical): 288 of the 1601 wavefronts per warp leave the L1 data
// pipe, and the kernel is SLOWER, 2.94 ms against 2.84 ms at 48^3x96 -- with the wait placed right behind the load 2.97 ms:
// LDTM moves 64 B/clk per SM, half of what the data pipe does, so the 16 own-link fetches per site cost 576 clocks per
// warp there, and tcgen05.wait::ld waits for all of a thread's outstanding loads.  Kept as an option and as the measurement.
__device__ __forceinline__ void tmem_store_mat(unsigned taddr, const Mat3<float>& m) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
                 "f"(m.re[0][0]), "f"(m.im[0][0]), "f"(m.re[0][1]), "f"(m.im[0][1]), "f"(m.re[0][2]), "f"(m.im[0][2]), "f"(m.re[1][0]),
                 "f"(m.im[1][0]), "f"(m.re[1][1]), "f"(m.im[1][1]), "f"(m.re[1][2]), "f"(m.im[1][2]), "f"(m.re[2][0]), "f"(m.im[2][0]),
                 "f"(m.re[2][1]), "f"(m.im[2][1]));
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1,%2};" ::"r"(taddr + 16), "f"(m.re[2][2]), "f"(m.im[2][2]));
}
__device__ __forceinline__ Mat3<float> tmem_load_mat(unsigned taddr) {
    Mat3<float> m;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=f"(m.re[0][0]), "=f"(m.im[0][0]), "=f"(m.re[0][1]), "=f"(m.im[0][1]), "=f"(m.re[0][2]), "=f"(m.im[0][2]), "=f"(m.re[1][0]),
                   "=f"(m.im[1][0]), "=f"(m.re[1][1]), "=f"(m.im[1][1]), "=f"(m.re[1][2]), "=f"(m.im[1][2]), "=f"(m.re[2][0]), "=f"(m.im[2][0]),
                   "=f"(m.re[2][1]), "=f"(m.im[2][1])
                 : "r"(taddr));
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=f"(m.re[2][2]), "=f"(m.im[2][2]) : "r"(taddr + 16));
    return m;  // NOT valid before tmem_wait(m)
}
// the loaded registers pass through the wait as in/out operands, so that no use of them can be scheduled above it
__device__ __forceinline__ void tmem_wait(Mat3<float>& m) {
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+f"(m.re[0][0]), "+f"(m.im[0][0]), "+f"(m.re[0][1]), "+f"(m.im[0][1]), "+f"(m.re[0][2]), "+f"(m.im[0][2]), "+f"(m.re[1][0]),
                   "+f"(m.im[1][0]), "+f"(m.re[1][1]), "+f"(m.im[1][1]), "+f"(m.re[1][2]), "+f"(m.im[1][2]), "+f"(m.re[2][0]), "+f"(m.im[2][0]),
                   "+f"(m.re[2][1]), "+f"(m.im[2][1]), "+f"(m.re[2][2]), "+f"(m.im[2][2]));
}
constexpr int kTmemCols = 256;  // per CTA: three warps per lane quarter x 72 words; two CTAs per SM use all 512 columns

// --------------------------------------------------------------------------------------------------------------
// Variant 9: the LITERAL evaluation (rolled loops, 48 products, the summation order of k_smear_rolled -- bit-identical
// to it) on the same whole-x-row tiles: 80 registers, two 384-thread CTAs per SM (24 warps, each CTA's fill overlaps the
// other's products), the tile's own links in shared memory, the halo through L2.
// Tried on top of it and dropped: the 24 staples with compile-time directions as the cases of a switch inside a rolled
// loop (a third fewer integer instructions, no spills -- but 4 000 instructions of straight-line code per site instead of
// 900 in loops, and with 24 warps at different places the instruction cache misses: 3.88 ms against 2.84 ms).
// --------------------------------------------------------------------------------------------------------------
// type shims so that the kernel template compiles for double, where tensor memory is not used (TM = false)
template <typename T>
__device__ __forceinline__ Mat3<T> tmem_own(unsigned taddr);
template <>
__device__ __forceinline__ Mat3<float> tmem_own<float>(unsigned taddr) { return tmem_load_mat(taddr); }
template <>
__device__ __forceinline__ Mat3<double> tmem_own<double>(unsigned) { return zero_mat<double>(); }
__device__ __forceinline__ void tmem_put(unsigned taddr, const Mat3<float>& m) { tmem_store_mat(taddr, m); }
__device__ __forceinline__ void tmem_put(unsigned, const Mat3<double>&) {}
__device__ __forceinline__ void tmem_wait_t(Mat3<float>& m) { tmem_wait(m); }
__device__ __forceinline__ void tmem_wait_t(Mat3<double>&) {}

template <typename T, bool PLAQ, int RY, int RZ, int RT, int MAXT, int MINB, bool TM, bool BULK>
__global__ void __launch_bounds__(MAXT, MINB) k_smear_rowlit(const __grid_constant__ Geo g, const __grid_constant__ RowMap rm,
                                                          const __grid_constant__ Links<T> u, const __grid_constant__ LinksOut<T> out,
                                                          T c0, T c1, double* __restrict__ partials) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int L0 = g.L[0];
    const int nthr = blockDim.x;
    const int npad = (nthr + 31) & ~31;
    const int link_floats = 18 * npad;
    T* const buf0 = reinterpret_cast<T*>(smem_raw);
    const int li = threadIdx.x;
    const int lx = li % L0, row = li / L0;
    const int ly = row % RY, lz = (row / RY) % RZ, lt = row / (RY * RZ);
    int x[4];
    int s;
    {
        const int tile = blockIdx.x;
        const int per_slab = rm.ny * rm.zs * rm.nt;
        const int k = tile / per_slab;
        int rem = tile - k * per_slab;
        const int bt = rem / (rm.ny * rm.zs);
        rem -= bt * (rm.ny * rm.zs);
        const int bz = rem / rm.ny + k * rm.zs, by = rem % rm.ny;
        x[0] = lx, x[1] = RY * by + ly, x[2] = RZ * bz + lz, x[3] = RT * (bt + rm.toff) + lt;
        s = x[0] + g.L[0] * (x[1] + g.L[1] * (x[2] + g.L[2] * x[3]));
    }
    __shared__ __align__(8) unsigned long long fill_bar;  // referenced by the BULK instantiations only
    const unsigned bar = BULK ? (unsigned)__cvta_generic_to_shared(&fill_bar) : 0u;
    if (BULK) {
        if (li == 0) mbar_init(bar, 1);
        __syncthreads();
        if (li < 32) {
            // group k = (lz, lt): RY rows = grp_reals reals per link, contiguous in the field and in the tile buffer
            const int grp_sites = RY * L0;
            const unsigned grp_bytes = (unsigned)(grp_sites * 18 * sizeof(T));
            if (li == 0) mbar_expect(bar, grp_bytes * (RZ * RT * 4));
            __syncwarp();
            // the site of lane 0's thread is the tile's first site: s0 = s - li is the first site of group 0
            const int s0 = __shfl_sync(0xffffffffu, s, 0);
            for (int c = li; c < RZ * RT * 4; c += 32) {
                const int k = c >> 2, mu = c & 3;
                const int kz = k % RZ, kt = k / RZ;
                const int sk = s0 + g.L[0] * g.L[1] * (kz + g.L[2] * kt);
                bulk_g2s((unsigned)__cvta_generic_to_shared(buf0 + mu * link_floats + k * grp_sites * 18),
                         u.u[mu] + (size_t)(sk >> 5) * (32 * 18), grp_bytes, bar);
            }
        }
    } else {
        fill_async(buf0, link_floats, u, s, li);
    }
    __pipeline_commit();
    unsigned mask = (ly + 1 < RY ? 2u : 0u) | (lz + 1 < RZ ? 4u : 0u) | (lt + 1 < RT ? 8u : 0u) | (ly > 0 ? 32u : 0u) |
                    (lz > 0 ? 64u : 0u) | (lt > 0 ? 128u : 0u) | 17u;  // x-neighbours are always in the tile
#pragma unroll
    for (int d = 0; d < 4; ++d) {
        if (x[d] + 1 == g.L[d]) mask |= 1u << (8 + d);
        if (x[d] == 0) mask |= 1u << (12 + d);
    }
    const int dpx = (lx + 1 == L0) ? -(L0 - 1) : 1, dmx = (lx == 0) ? (L0 - 1) : -1;
    // tile-local index delta, global site index of a neighbour, for a run-time direction
    auto dloc = [&](int d, bool fwd) {
        const int r = d == 1 ? L0 : (d == 2 ? RY * L0 : RY * RZ * L0);
        return d == 0 ? (fwd ? dpx : dmx) : (fwd ? r : -r);
    };
    auto gnb = [&](int d, bool fwd) {
        const int wrap = (g.L[d] - 1) * g.stride_site[d];
        if (fwd) return ((mask >> (8 + d)) & 1u) ? s - wrap : s + g.stride_site[d];
        return ((mask >> (12 + d)) & 1u) ? s + wrap : s - g.stride_site[d];
    };
    __shared__ unsigned tm_base_s;
    if (TM && (li >> 5) == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(&tm_base_s)),
                     "n"(kTmemCols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    if (BULK) mbar_wait(bar, 0);
    else __pipeline_wait_prior(0);
    if (TM) asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    unsigned tm_own = 0;  // TMEM address of this thread's U_0(x): lane quarter of the warp, 72 columns per warp of a quarter
    if (TM) {
        asm volatile("tcgen05.fence::after_thread_sync;");
        const int w = li >> 5;
        tm_own = tm_base_s + ((unsigned)((w & 3) * 32) << 16) + (unsigned)((w >> 2) * 72);
#pragma unroll 1
        for (int mu = 0; mu < 4; ++mu) tmem_put(tm_own + 18 * mu, fetch_own_t<T>((unsigned long long)(buf0 + mu * link_floats), li));
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }

    T pl = T(0);
#pragma unroll 1
    for (int mu = 0; mu < 4; ++mu) {
        const T* umu_g = u.u[mu];
        const unsigned long long umu_t = (unsigned long long)(buf0 + mu * link_floats);
        const int xpmu = gnb(mu, true);
        const bool in_pmu = (mask >> mu) & 1u;
        const int d_pmu = dloc(mu, true);
        Mat3<T> acc = zero_mat<T>();
#pragma unroll 1
        for (int nu = 3; nu >= 0; --nu) {  // upper: U_nu(x) U_mu(x+nu^) adj(U_nu(x+mu^))
            if (nu == mu) continue;
            const T* unu_g = u.u[nu];
            const unsigned long long unu_t = (unsigned long long)(buf0 + nu * link_floats);
            const bool in_pnu = (mask >> nu) & 1u;
            Mat3<T> own = TM ? tmem_own<T>(tm_own + 18 * nu) : fetch_own_t<T>(unu_t, li);  // requested first, awaited last
            const Mat3<T> second = fetch_mat(umu_t, umu_g, in_pnu, li + dloc(nu, true), gnb(nu, true));
            if (TM) tmem_wait_t(own);
            const Mat3<T> t = mul_nn(own, second);
            mac_na(acc, t, fetch_mat(unu_t, unu_g, in_pmu, li + d_pmu, xpmu));
        }
#pragma unroll 1
        for (int nu = 0; nu < 4; ++nu) {  // lower: adj(U_nu(x-nu^)) U_mu(x-nu^) U_nu(x-nu^+mu^)
            if (nu == mu) continue;
            const T* unu_g = u.u[nu];
            const unsigned long long unu_t = (unsigned long long)(buf0 + nu * link_floats);
            const bool in_mnu = (mask >> (4 + nu)) & 1u;
            const int xmnu = gnb(nu, false);
            const int l1 = li + dloc(nu, false);
            const Mat3<T> t = mul_an(fetch_mat(unu_t, unu_g, in_mnu, l1, xmnu), fetch_mat(umu_t, umu_g, in_mnu, l1, xmnu));
            mac_nn(acc, t, fetch_mat(unu_t, unu_g, in_mnu && in_pmu, l1 + d_pmu, xmnu + (xpmu - s)));
        }
        Mat3<T> umu = TM ? tmem_own<T>(tm_own + 18 * mu) : fetch_own_t<T>(umu_t, li);
        if (TM) tmem_wait_t(umu);
        if (PLAQ) pl += re_tr_na(umu, acc);
        Mat3<T> r;
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                r.re[i][j] = fma(c1, acc.re[i][j], c0 * umu.re[i][j]);
                r.im[i][j] = fma(c1, acc.im[i][j], c0 * umu.im[i][j]);
            }
        store_mat_cs(out.u[mu], s, r);
    }
    if (PLAQ) {
        double p[1] = {0.25 * (double)pl};
        block_reduce_partial<1>(p, partials);
    }
    if (TM) {  // every warp is done with its columns before warp 0 gives them back
        asm volatile("tcgen05.fence::before_thread_sync;");
        __syncthreads();
        if ((li >> 5) == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tm_base_s), "n"(kTmemCols));
    }
}

// --------------------------------------------------------------------------------------------------------------
// Variant 10: the per-link evaluation of variant 9 with the upper staples' common factor kept in TENSOR MEMORY.
// For a plane a < b the product Z'_ab = U_a(x+b^) adj(U_b(x+a^)) serves the upper staple of link a, U_b(x) Z'_ab, and of
// link b, U_a(x) adj(Z'_ab).  Variant 8 uses this with all four staple sums live (168 registers, 12 warps per SM); here the
// links are still processed one after the other with ONE accumulator (80 registers, 24 warps), and Z'_ab waits in the
// thread's own TMEM lane from link a to link b: at most four matrices = 72 columns per warp (tcgen05.st / tcgen05.ld as a
// per-thread scratchpad, no tensor-core instruction).  42 products and 64 operand fetches per site instead of 48 / 76, the
// six saved operand pairs being neighbour fetches; in exchange 6 x 18 words written to and read from TMEM (256 / 64 B/clk).
// The nu loop runs ASCENDING here (nu < mu consumes, nu > mu produces, so a slot is free before it is needed again) and the
// upper staple is associated as U_nu(x) (U_mu(x+nu^) adj(U_nu(x+mu^))): agrees with the other variants to rounding.
// Eight-row tiles only (three warps per TMEM lane quarter x 72 columns = 216 of the CTA's 256 columns; two CTAs per SM).
// --------------------------------------------------------------------------------------------------------------
template <bool PLAQ, int RY, int RZ, int RT, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) k_smear_rowz(const __grid_constant__ Geo g, const __grid_constant__ RowMap rm,
                                                        const __grid_constant__ Links<float> u, const __grid_constant__ LinksOut<float> out,
                                                        float c0, float c1, double* __restrict__ partials) {
    typedef float T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int L0 = g.L[0];
    const int nthr = blockDim.x;
    const int npad = (nthr + 31) & ~31;
    const int link_floats = 18 * npad;
    T* const buf0 = reinterpret_cast<T*>(smem_raw);
    const int li = threadIdx.x;
    const int lx = li % L0, row = li / L0;
    const int ly = row % RY, lz = (row / RY) % RZ, lt = row / (RY * RZ);
    int x[4];
    int s;
    {
        const int tile = blockIdx.x;
        const int per_slab = rm.ny * rm.zs * rm.nt;
        const int k = tile / per_slab;
        int rem = tile - k * per_slab;
        const int bt = rem / (rm.ny * rm.zs);
        rem -= bt * (rm.ny * rm.zs);
        const int bz = rem / rm.ny + k * rm.zs, by = rem % rm.ny;
        x[0] = lx, x[1] = RY * by + ly, x[2] = RZ * bz + lz, x[3] = RT * (bt + rm.toff) + lt;
        s = x[0] + g.L[0] * (x[1] + g.L[1] * (x[2] + g.L[2] * x[3]));
    }
    fill_async(buf0, link_floats, u, s, li);
    __pipeline_commit();
    unsigned mask = (ly + 1 < RY ? 2u : 0u) | (lz + 1 < RZ ? 4u : 0u) | (lt + 1 < RT ? 8u : 0u) | (ly > 0 ? 32u : 0u) |
                    (lz > 0 ? 64u : 0u) | (lt > 0 ? 128u : 0u) | 17u;  // x-neighbours are always in the tile
#pragma unroll
    for (int d = 0; d < 4; ++d) {
        if (x[d] + 1 == g.L[d]) mask |= 1u << (8 + d);
        if (x[d] == 0) mask |= 1u << (12 + d);
    }
    const int dpx = (lx + 1 == L0) ? -(L0 - 1) : 1, dmx = (lx == 0) ? (L0 - 1) : -1;
    auto dloc = [&](int d, bool fwd) {
        const int r = d == 1 ? L0 : (d == 2 ? RY * L0 : RY * RZ * L0);
        return d == 0 ? (fwd ? dpx : dmx) : (fwd ? r : -r);
    };
    auto gnb = [&](int d, bool fwd) {
        const int wrap = (g.L[d] - 1) * g.stride_site[d];
        if (fwd) return ((mask >> (8 + d)) & 1u) ? s - wrap : s + g.stride_site[d];
        return ((mask >> (12 + d)) & 1u) ? s + wrap : s - g.stride_site[d];
    };
    __shared__ unsigned tm_base_s;
    // columns: 72 per warp of a lane quarter, rounded up to the power of two tcgen05.alloc takes
    const unsigned tm_need = (unsigned)(((nthr >> 5) + 3) >> 2) * 72u;
    const unsigned tm_cols = tm_need <= 128u ? 128u : 256u;
    if ((li >> 5) == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(&tm_base_s)),
                     "r"(tm_cols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    __pipeline_wait_prior(0);
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    // this thread's scratch: the lane quarter of its warp, 72 columns per warp of a quarter, four slots of 18 columns
    const unsigned tm_z = tm_base_s + ((unsigned)(((li >> 5) & 3) * 32) << 16) + (unsigned)((li >> 7) * 72);
    // slot of plane (a, b), a < b, packed two bits per entry at index 4 a + b: (0,1) 0, (0,2) 1, (0,3) 2, (1,2) 0, (1,3) 3, (2,3) 0
    constexpr unsigned kSlots = (0u << 2) | (1u << 4) | (2u << 6) | (0u << 12) | (3u << 14) | (0u << 22);

    T pl = T(0);
#pragma unroll 1
    for (int mu = 0; mu < 4; ++mu) {
        const T* umu_g = u.u[mu];
        const unsigned long long umu_t = (unsigned long long)(buf0 + mu * link_floats);
        const int xpmu = gnb(mu, true);
        const bool in_pmu = (mask >> mu) & 1u;
        const int d_pmu = dloc(mu, true);
        Mat3<T> acc = zero_mat<T>();
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");  // the factors stored while the earlier links were processed
#pragma unroll 1
        for (int nu = 0; nu < 4; ++nu) {  // upper: U_nu(x) [U_mu(x+nu^) adj(U_nu(x+mu^))]
            if (nu == mu) continue;
            const T* unu_g = u.u[nu];
            const unsigned long long unu_t = (unsigned long long)(buf0 + nu * link_floats);
            if (nu < mu) {  // the bracket is adj(Z'_{nu mu}), produced when link nu was processed
                const unsigned slot = (kSlots >> (2 * (4 * nu + mu))) & 3u;
                Mat3<T> z = tmem_load_mat(tm_z + 18 * slot);
                const Mat3<T> own = fetch_own(unu_t, li);
                tmem_wait(z);
                mac_na(acc, own, z);
            } else {  // produce Z'_{mu nu} and keep it for link nu
                const bool in_pnu = (mask >> nu) & 1u;
                const Mat3<T> second = fetch_mat(umu_t, umu_g, in_pnu, li + dloc(nu, true), gnb(nu, true));
                const Mat3<T> z = mul_na(second, fetch_mat(unu_t, unu_g, in_pmu, li + d_pmu, xpmu));
                const unsigned slot = (kSlots >> (2 * (4 * mu + nu))) & 3u;
                tmem_store_mat(tm_z + 18 * slot, z);
                mac_nn(acc, fetch_own(unu_t, li), z);
            }
        }
#pragma unroll 1
        for (int nu = 0; nu < 4; ++nu) {  // lower: adj(U_nu(x-nu^)) U_mu(x-nu^) U_nu(x-nu^+mu^)
            if (nu == mu) continue;
            const T* unu_g = u.u[nu];
            const unsigned long long unu_t = (unsigned long long)(buf0 + nu * link_floats);
            const bool in_mnu = (mask >> (4 + nu)) & 1u;
            const int xmnu = gnb(nu, false);
            const int l1 = li + dloc(nu, false);
            const Mat3<T> t = mul_an(fetch_mat(unu_t, unu_g, in_mnu, l1, xmnu), fetch_mat(umu_t, umu_g, in_mnu, l1, xmnu));
            mac_nn(acc, t, fetch_mat(unu_t, unu_g, in_mnu && in_pmu, l1 + d_pmu, xmnu + (xpmu - s)));
        }
        const Mat3<T> umu = fetch_own(umu_t, li);
        if (PLAQ) pl += re_tr_na(umu, acc);
        Mat3<T> r;
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                r.re[i][j] = fma(c1, acc.re[i][j], c0 * umu.re[i][j]);
                r.im[i][j] = fma(c1, acc.im[i][j], c0 * umu.im[i][j]);
            }
        store_mat_cs(out.u[mu], s, r);
    }
    if (PLAQ) {
        double p[1] = {0.25 * (double)pl};
        block_reduce_partial<1>(p, partials);
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if ((li >> 5) == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tm_base_s), "r"(tm_cols));
}

// t0 < 0: the whole lattice; otherwise the time slices [t0, t1) only (both multiples of RT; no plaquette)
template <int RY, int RZ, int RT, int MAXT, int MINB>
int rowz_launch(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, double* plaq, int t0 = -1, int t1 = -1) {
    const Geo& g = ctx->geo;
    const int nthr = g.L[0] * RY * RZ * RT;
    // whole warps, and at most three warps per TMEM lane quarter (72 columns each of the CTA's 256)
    if (nthr > MAXT || nthr % 32 || nthr > 384 || g.L[1] % RY || g.L[2] % RZ || g.L[3] % RT || (size_t)g.Vpad * 72 >= ((size_t)1 << 32)) return 1;
    if (t0 >= 0 && (t0 % RT || t1 % RT || plaq)) return 1;
    RowMap rm;
    rm.ny = g.L[1] / RY, rm.nz = g.L[2] / RZ, rm.nt = t0 >= 0 ? (t1 - t0) / RT : g.L[3] / RT;
    rm.toff = t0 >= 0 ? t0 / RT : 0;
    rm.ntiles = rm.ny * rm.nz * rm.nt;
    int target = ctx->opt_block > 0 ? ctx->opt_block : kSlabZ;
    rm.zs = 1;
    for (int z = 1; z <= rm.nz; ++z)
        if (rm.nz % z == 0 && z * RZ <= target) rm.zs = z;
    const int npad = (nthr + 31) & ~31;
    const size_t smem = (size_t)4 * 18 * npad * sizeof(float);
    const int grid = rm.ntiles;
    if (plaq) LQX_CUDA(ctx, cudaFuncSetAttribute(k_smear_rowz<true, RY, RZ, RT, MAXT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    else LQX_CUDA(ctx, cudaFuncSetAttribute(k_smear_rowz<false, RY, RZ, RT, MAXT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (plaq) {
        int rc = lqx_ensure_partials(ctx, (size_t)grid);
        if (rc) return rc;
    }
    {
        LqxTimed timed(ctx, LQX_K_SMEAR);
        if (plaq) k_smear_rowz<true, RY, RZ, RT, MAXT, MINB><<<grid, nthr, smem, ctx->stream>>>(g, rm, in, out, c0, c1, ctx->d_partials);
        else k_smear_rowz<false, RY, RZ, RT, MAXT, MINB><<<grid, nthr, smem, ctx->stream>>>(g, rm, in, out, c0, c1, nullptr);
    }
    LQX_LAUNCH_CHECK(ctx);
    return plaq ? lqx_sum_partials(ctx, grid, 1, plaq) : LQX_OK;
}

// t0 < 0: the whole lattice; otherwise the time slices [t0, t1) only (both multiples of RT, else 1; no plaquette)
template <typename T, int RY, int RZ, int RT, int MAXT, int MINB, bool TM = false, bool BULK = false>
int rowlit_launch(lqx_ctx* ctx, const Links<T>& in, const LinksOut<T>& out, T c0, T c1, double* plaq,
                  int t0 = -1, int t1 = -1) {
    const Geo& g = ctx->geo;
    const int nthr = g.L[0] * RY * RZ * RT;
    // whole warps only: the CTA-wide reductions shuffle with a full mask
    if (nthr > MAXT || nthr % 32 || g.L[1] % RY || g.L[2] % RZ || g.L[3] % RT || (size_t)g.Vpad * 18 * sizeof(T) >= ((size_t)1 << 32)) return 1;
    if (t0 >= 0 && (t0 % RT || t1 % RT || plaq)) return 1;
    RowMap rm;
    rm.ny = g.L[1] / RY, rm.nz = g.L[2] / RZ, rm.nt = t0 >= 0 ? (t1 - t0) / RT : g.L[3] / RT;
    rm.toff = t0 >= 0 ? t0 / RT : 0;
    rm.ntiles = rm.ny * rm.nz * rm.nt;
    if (BULK && (RY * g.L[0]) % 32 != 0) return 1;
    int target = ctx->opt_block > 0 ? ctx->opt_block : kSlabZ;
    rm.zs = 1;
    for (int z = 1; z <= rm.nz; ++z)
        if (rm.nz % z == 0 && z * RZ <= target) rm.zs = z;
    const int npad = (nthr + 31) & ~31;
    const size_t smem = (size_t)4 * 18 * npad * sizeof(T);
    const int grid = rm.ntiles;
    if (plaq) LQX_CUDA(ctx, cudaFuncSetAttribute(k_smear_rowlit<T, true, RY, RZ, RT, MAXT, MINB, TM, BULK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    else LQX_CUDA(ctx, cudaFuncSetAttribute(k_smear_rowlit<T, false, RY, RZ, RT, MAXT, MINB, TM, BULK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (plaq) {
        int rc = lqx_ensure_partials(ctx, (size_t)grid);
        if (rc) return rc;
    }
    {
        LqxTimed timed(ctx, LQX_K_SMEAR);
        if (plaq) k_smear_rowlit<T, true, RY, RZ, RT, MAXT, MINB, TM, BULK><<<grid, nthr, smem, ctx->stream>>>(g, rm, in, out, c0, c1, ctx->d_partials);
        else k_smear_rowlit<T, false, RY, RZ, RT, MAXT, MINB, TM, BULK><<<grid, nthr, smem, ctx->stream>>>(g, rm, in, out, c0, c1, nullptr);
    }
    LQX_LAUNCH_CHECK(ctx);
    return plaq ? lqx_sum_partials(ctx, grid, 1, plaq) : LQX_OK;
}

template <int RY, int RZ, int RT, int MAXT, int MINB = 1, bool PF = false>
int rows_launch(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, double* plaq) {
    const Geo& g = ctx->geo;
    const int nthr = g.L[0] * RY * RZ * RT;
    // whole warps only: the CTA-wide reductions shuffle with a full mask
    if (nthr > MAXT || nthr % 32 || g.L[1] % RY || g.L[2] % RZ || g.L[3] % RT || (size_t)g.Vpad * 72 >= ((size_t)1 << 32)) return 1;
    RowMap rm;
    rm.ny = g.L[1] / RY, rm.nz = g.L[2] / RZ, rm.nt = g.L[3] / RT;
    rm.toff = 0;
    rm.ntiles = rm.ny * rm.nz * rm.nt;
    // slab thickness in z: the largest divisor of nz that keeps a slab at most kSlabZ sites thick
    int target = ctx->opt_block > 0 ? ctx->opt_block : kSlabZ;
    rm.zs = 1;
    for (int z = 1; z <= rm.nz; ++z)
        if (rm.nz % z == 0 && z * RZ <= target) rm.zs = z;
    const int npad = (nthr + 31) & ~31;
    // MINB = 1: persistent CTAs, one per SM, two tile buffers (the next tile's links arrive during this tile's products).
    // MINB > 1: one tile per CTA and one buffer, MINB CTAs per SM; what is left of the SM's 256 KB stays L1 for the halo.
    const size_t smem = (MINB == 1 ? 2 : 1) * (size_t)4 * 18 * npad * sizeof(float);
    if (smem > 227 * 1024) return 1;
    const int grid = MINB == 1 ? std::min(rm.ntiles, ctx->num_sms) : rm.ntiles;
    if (plaq) LQX_CUDA(ctx, cudaFuncSetAttribute(k_smear_rows<true, RY, RZ, RT, MAXT, MINB, PF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    else LQX_CUDA(ctx, cudaFuncSetAttribute(k_smear_rows<false, RY, RZ, RT, MAXT, MINB, PF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (plaq) {
        int rc = lqx_ensure_partials(ctx, (size_t)grid);
        if (rc) return rc;
    }
    {
        LqxTimed timed(ctx, LQX_K_SMEAR);
        if (plaq) k_smear_rows<true, RY, RZ, RT, MAXT, MINB, PF><<<grid, nthr, smem, ctx->stream>>>(g, rm, in, out, c0, c1, ctx->d_partials);
        else k_smear_rows<false, RY, RZ, RT, MAXT, MINB, PF><<<grid, nthr, smem, ctx->stream>>>(g, rm, in, out, c0, c1, nullptr);
    }
    LQX_LAUNCH_CHECK(ctx);
    return plaq ? lqx_sum_partials(ctx, grid, 1, plaq) : LQX_OK;
}

}  // namespace

// LQX_OK, a negative status, or 1 if the lattice does not fit this kernel.  Option "tile" picks the rows of a tile:
// 1 = 2x3x1 (y, z, t; 6 rows), 2 = 3x2x1, 3 = 2x2x2 (8 rows), 4 = 2x1x3, 5 = 1x2x3; automatic = the first that fits;
// 6 = 2x2x1 rows, one tile per CTA, two CTAs per SM; 7 = 6 with the halo operands prefetched into L1
int lqx_smear_rows_launch(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, double* plaq) {
    const int t = ctx->opt_tile;
    int rc = 1;
    if (t == 1 || t <= 0) rc = rows_launch<2, 3, 1, 288>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t == 2 || t <= 0) rc = rows_launch<3, 2, 1, 288>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t == 3 || t <= 0) rc = rows_launch<2, 2, 2, 384>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t == 4) rc = rows_launch<2, 1, 3, 288>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t == 5) rc = rows_launch<1, 2, 3, 288>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t == 6) rc = rows_launch<2, 2, 1, 192, 2, false>(ctx, in, out, c0, c1, plaq);  // two CTAs per SM, L1 left for the halo
    if (rc != 1) return rc;
    if (t == 7) rc = rows_launch<2, 2, 1, 192, 2, true>(ctx, in, out, c0, c1, plaq);   // ... with L1 prefetch of the halo operands
    return rc;
}

// variant 9 (literal evaluation on row tiles).  Option "tile": 1 = 2x2x2 rows (8, the default), 2 = 2x2x1 rows four CTAs per SM,
// 3 = 2x2x1 three CTAs (96 registers), 4 = 2x3x1, 5 = 3x2x1, 6 = 2x2x2 one CTA per SM (128 registers),
// 7 = 2x2x2 with the own links re-read from tensor memory
int lqx_smear_rowlit_launch(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, double* plaq) {
    const int t = ctx->opt_tile;
    int rc = 1;
    const bool bulk = ctx->opt_bulk_fill > 0;  // tiles 1 and 2 only; 1 = not applicable (rows are not whole blocks): cp.async
    if (bulk && (t == 1 || t <= 0)) rc = rowlit_launch<float, 2, 2, 2, 384, 2, false, true>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t == 1 || t <= 0) rc = rowlit_launch<float, 2, 2, 2, 384, 2>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (bulk && (t == 2 || t <= 0)) rc = rowlit_launch<float, 2, 2, 1, 192, 4, false, true>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t == 2 || t <= 0) rc = rowlit_launch<float, 2, 2, 1, 192, 4>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t <= 0) rc = rowlit_launch<float, 2, 2, 1, 384, 2>(ctx, in, out, c0, c1, plaq);  // rows of 49 .. 96 sites: four-row tiles
    if (rc != 1) return rc;
    if (t == 3) rc = rowlit_launch<float, 2, 2, 1, 192, 3>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t == 4) rc = rowlit_launch<float, 2, 3, 1, 288, 2>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t == 5) rc = rowlit_launch<float, 3, 2, 1, 288, 2>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t == 6) rc = rowlit_launch<float, 2, 2, 2, 384, 1>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t == 7) rc = rowlit_launch<float, 2, 2, 2, 384, 2, true>(ctx, in, out, c0, c1, plaq);  // own links re-read from tensor memory
    return rc;
}

// the default fp32 kernel on the time slices [t0, t1) only: LQX_OK, a negative status, or 1 if the row tiles do not
// fit the lattice or do not split at t0 / t1 (the caller then launches the rolled kernel, which is bit-identical)
int lqx_smear_rowlit_launch_range(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, int t0, int t1) {
    return rowlit_launch<float, 2, 2, 2, 384, 2>(ctx, in, out, c0, c1, nullptr, t0, t1);
}

// variant 9 in double precision: four-row tiles (L0 x 2 x 2 x 1 sites; 72 KB of shared memory at L0 = 32), as many CTAs per
// SM as the 168 registers of the fp64 literal evaluation allow.  Option "tile": 1 = 2x2x1 rows, 2 = 2x1x2, 3 = 2x2x2
int lqx_smear_rowlit_launch(lqx_ctx* ctx, const Links<double>& in, const LinksOut<double>& out, double c0, double c1, double* plaq) {
    const int t = ctx->opt_tile;
    int rc = 1;
    if (ctx->opt_bulk_fill > 0 && (t == 1 || t <= 0)) rc = rowlit_launch<double, 2, 2, 1, 128, 3, false, true>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t == 1 || t <= 0) rc = rowlit_launch<double, 2, 2, 1, 128, 3>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t == 2) rc = rowlit_launch<double, 2, 1, 2, 128, 3>(ctx, in, out, c0, c1, plaq);
    if (rc != 1) return rc;
    if (t == 3) rc = rowlit_launch<double, 2, 2, 2, 256, 1>(ctx, in, out, c0, c1, plaq);
    return rc;
}

// variant 10 (upper-staple factors kept in tensor memory; fp32).  It runs where a row pair is whole warps and a tile at most
// 384 threads (L0 a multiple of 8, at most 48; L1, L2 even): eight-row tiles, four-row tiles where a t-range or the
// lattice's t-extent is odd -- every tile shape evaluates the same per-site arithmetic.
bool lqx_smear_rowz_fits(const lqx_ctx* ctx) {
    const Geo& g = ctx->geo;
    return g.L[0] % 8 == 0 && g.L[0] * 8 <= 384 && g.L[1] % 2 == 0 && g.L[2] % 2 == 0;
}
// LQX_OK, a negative status, or 1 if the lattice does not fit (the caller falls back to variant 9)
int lqx_smear_rowz_launch(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, double* plaq) {
    if (!lqx_smear_rowz_fits(ctx)) return 1;
    if (ctx->geo.L[3] % 2 == 0) return rowz_launch<2, 2, 2, 384, 2>(ctx, in, out, c0, c1, plaq);
    return rowz_launch<2, 2, 1, 192, 2>(ctx, in, out, c0, c1, plaq);
}
int lqx_smear_rowz_launch_range(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, int t0, int t1) {
    if (!lqx_smear_rowz_fits(ctx)) return 1;
    if (t0 % 2 == 0 && t1 % 2 == 0 && ctx->geo.L[3] % 2 == 0) return rowz_launch<2, 2, 2, 384, 2>(ctx, in, out, c0, c1, nullptr, t0, t1);
    return rowz_launch<2, 2, 1, 192, 2>(ctx, in, out, c0, c1, nullptr, t0, t1);
}
