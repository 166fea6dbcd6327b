// lqx staple sum + smear step, shared-memory-staged variant (option "smear_variant" = 6, fp32).
//
// The literal evaluation fetches 76 operand matrices per site through the L1 data pipe, 38 % of them L1 hits,
// and 45 % of its warp samples wait on those loads (profiles/r01c_smear_rolled.md).  Here one persistent CTA per
// SM walks over 8x2x2x2 tiles (64 sites); the ~1080 distinct link matrices a tile needs (the tile, its faces
// and the edges x-nu^+mu^) are copied global -> shared with cp.async into one of two buffers WHILE the CTA
// multiplies the previous tile out of the other buffer, so that operand latency no longer depends on occupancy
// and every later fetch is an aligned shared-memory read.  Four threads per site (one per link, as in
// k_smear_mu4): 256 threads, thread (site l, mu) adds its six staples in the order of k_smear_rolled, so the
// two kernels agree bit for bit.
// Two tables, built on the host for the tile shape and kept in device memory by the context:
//   footprint[slot]        = (dx+1) | (dy+1)<<4 | (dz+1)<<8 | (dt+1)<<12 | link<<16    what each slot holds
//   operand[(l*4+mu)*19+j] = slot of the j-th operand of thread (l, mu): 6 staples x 3 factors, then U_mu(x)
#include <cuda_pipeline.h>

#include <map>
#include <mutex>
#include <tuple>

#include "lqx_smear.cuh"

namespace {

constexpr int TX = 8, TY = 2, TZ = 2, TT = 2, NSITE = TX * TY * TZ * TT;  // 64 sites per tile
constexpr int NTHREADS = 4 * NSITE;                                      // 256
constexpr int SLOT_FLOATS = 20;                                          // 18 used: 80-byte slots are bank-conflict-free for LDS.128

__host__ __device__ inline int nu_upper(int mu, int k) {  // nu = 3, 2, 1, 0 without mu
    const int nu = 3 - k;
    return nu <= mu ? nu - 1 : nu;
}
__host__ __device__ inline int nu_lower(int mu, int k) {  // nu = 0, 1, 2, 3 without mu
    return k >= mu ? k + 1 : k;
}

struct StagedTables {
    int nslots = 0;
    std::vector<int> footprint;
    std::vector<unsigned short> operand;
};

// enumerate what thread (l, mu) reads, in the order it reads it, and number the distinct (link, offset) pairs
StagedTables build_tables() {
    const int T[4] = {TX, TY, TZ, TT};
    typedef std::tuple<int, int, int, int, int> Key;  // link, dt, dz, dy, dx  (x fastest inside a link: contiguous runs)
    std::map<Key, int> slot_of;
    std::vector<std::vector<Key>> want(NSITE * 4);
    for (int l = 0; l < NSITE; ++l) {
        const int x[4] = {l % TX, (l / TX) % TY, (l / (TX * TY)) % TZ, l / (TX * TY * TZ)};
        for (int mu = 0; mu < 4; ++mu) {
            std::vector<Key>& w = want[l * 4 + mu];
            auto key = [&](int link, int d0, int s0, int d1, int s1) {
                int y[4] = {x[0], x[1], x[2], x[3]};
                if (d0 >= 0) y[d0] += s0;
                if (d1 >= 0) y[d1] += s1;
                return Key(link, y[3], y[2], y[1], y[0]);
            };
            for (int k = 0; k < 3; ++k) {  // upper: U_nu(x) U_mu(x+nu^) adj(U_nu(x+mu^))
                const int nu = nu_upper(mu, k);
                w.push_back(key(nu, -1, 0, -1, 0));
                w.push_back(key(mu, nu, +1, -1, 0));
                w.push_back(key(nu, mu, +1, -1, 0));
            }
            for (int k = 0; k < 3; ++k) {  // lower: adj(U_nu(x-nu^)) U_mu(x-nu^) U_nu(x-nu^+mu^)
                const int nu = nu_lower(mu, k);
                w.push_back(key(nu, nu, -1, -1, 0));
                w.push_back(key(mu, nu, -1, -1, 0));
                w.push_back(key(nu, nu, -1, mu, +1));
            }
            w.push_back(key(mu, -1, 0, -1, 0));  // U_mu(x) for the update and the plaquette term
            for (const Key& kk : w) slot_of[kk] = 0;
        }
    }
    StagedTables t;
    for (auto& kv : slot_of) {  // std::map iterates in key order: link, t, z, y, x
        kv.second = t.nslots++;
        const Key& k = kv.first;
        t.footprint.push_back((std::get<4>(k) + 1) | ((std::get<3>(k) + 1) << 4) | ((std::get<2>(k) + 1) << 8) |
                              ((std::get<1>(k) + 1) << 12) | (std::get<0>(k) << 16));
    }
    t.operand.resize((size_t)NSITE * 4 * 19);
    for (int i = 0; i < NSITE * 4; ++i)
        for (int j = 0; j < 19; ++j) t.operand[(size_t)i * 19 + j] = (unsigned short)slot_of[want[i][j]];
    (void)T;
    return t;
}
// tile id -> tile origin, in the slab order of Tiled<>::site (x, y, z fastest inside a slab of zs z-tiles, then t)
__device__ __forceinline__ void tile_origin(const TileMap& m, int id, int org[4]) {
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
    org[0] = tx * TX;
    org[1] = ty * TY;
    org[2] = (tz + k * m.zs) * TZ;
    org[3] = tt * TT;
}

__device__ __forceinline__ Mat3<float> lds_mat(const float* __restrict__ slot) {
    const float4 a = reinterpret_cast<const float4*>(slot)[0], b = reinterpret_cast<const float4*>(slot)[1];
    const float4 c = reinterpret_cast<const float4*>(slot)[2], d = reinterpret_cast<const float4*>(slot)[3];
    const float2 e = reinterpret_cast<const float2*>(slot)[8];
    Mat3<float> m;
    m.re[0][0] = a.x; m.im[0][0] = a.y; m.re[0][1] = a.z; m.im[0][1] = a.w;
    m.re[0][2] = b.x; m.im[0][2] = b.y; m.re[1][0] = b.z; m.im[1][0] = b.w;
    m.re[1][1] = c.x; m.im[1][1] = c.y; m.re[1][2] = c.z; m.im[1][2] = c.w;
    m.re[2][0] = d.x; m.im[2][0] = d.y; m.re[2][1] = d.z; m.im[2][1] = d.w;
    m.re[2][2] = e.x; m.im[2][2] = e.y;
    return m;
}

template <bool PLAQ, int NBUF>
__global__ void __launch_bounds__(NTHREADS, 3 - NBUF) k_smear_staged(const __grid_constant__ Geo g, const __grid_constant__ TileMap tm,
                                                              const __grid_constant__ Links<float> u, const __grid_constant__ LinksOut<float> out,
                                                              float c0, float c1, int ntiles, int nslots, const int* __restrict__ footprint,
                                                              const unsigned short* __restrict__ operand, double* __restrict__ partials) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* buf0 = reinterpret_cast<float*>(smem_raw);
    float* buf1 = buf0 + (size_t)(NBUF - 1) * nslots * SLOT_FLOATS;  // == buf0 when single-buffered
    int* fp = reinterpret_cast<int*>(buf1 + (size_t)nslots * SLOT_FLOATS);
    unsigned short* op = reinterpret_cast<unsigned short*>(fp + nslots);
    const int tid = threadIdx.x;
    for (int j = tid; j < nslots; j += NTHREADS) fp[j] = footprint[j];
    for (int j = tid; j < NTHREADS * 19; j += NTHREADS) op[j] = operand[j];
    __syncthreads();

    // global -> shared copy of everything one tile needs (asynchronous: returns once the copies are issued)
    auto stage = [&](int tile, float* buf) {
        int org[4];
        tile_origin(tm, tile, org);
        for (int j = tid; j < nslots; j += NTHREADS) {
            const int f = fp[j];
            int c[4] = {org[0] + (f & 15) - 1, org[1] + ((f >> 4) & 15) - 1, org[2] + ((f >> 8) & 15) - 1, org[3] + ((f >> 12) & 15) - 1};
#pragma unroll
            for (int d = 0; d < 4; ++d) c[d] = c[d] < 0 ? c[d] + g.L[d] : (c[d] >= g.L[d] ? c[d] - g.L[d] : c[d]);
            const int s = c[0] + g.L[0] * (c[1] + g.L[1] * (c[2] + g.L[2] * c[3]));
            const float* blk = u.u[f >> 16] + (size_t)(s >> 5) * (32 * 18);
            const float* src = blk + (s & 31) * 4;
            float* dst = buf + (size_t)j * SLOT_FLOATS;
#pragma unroll
            for (int q = 0; q < 4; ++q) __pipeline_memcpy_async(dst + 4 * q, src + 128 * q, 16);
            __pipeline_memcpy_async(dst + 16, blk + 512 + (s & 31) * 2, 8);
        }
    };

    const int l = tid & (NSITE - 1), mu = tid / NSITE;
    const int lx[4] = {l % TX, (l / TX) % TY, (l / (TX * TY)) % TZ, l / (TX * TY * TZ)};
    const unsigned short* myop = op + (size_t)(l * 4 + mu) * 19;
    double plsum = 0.0;
    // NBUF = 2: the copies of the next tile are in flight while this one is multiplied (one CTA per SM);
    // NBUF = 1: stage, wait, multiply -- two CTAs per SM overlap each other instead
    int tile = blockIdx.x, i = 0;
    if (NBUF == 2) {
        if (tile < ntiles) stage(tile, buf0);
        __pipeline_commit();
    }
    for (; tile < ntiles; tile += gridDim.x, ++i) {
        float* cur = (NBUF == 2 && (i & 1)) ? buf1 : buf0;
        if (NBUF == 2) {
            const int next = tile + gridDim.x;
            if (next < ntiles) stage(next, (i & 1) ? buf0 : buf1);
            __pipeline_commit();
            __pipeline_wait_prior(1);  // everything but the copies just issued has landed: this tile is staged
        } else {
            stage(tile, buf0);
            __pipeline_commit();
            __pipeline_wait_prior(0);
        }
        __syncthreads();
        {
            Mat3<float> acc = zero_mat<float>();
#pragma unroll 1
            for (int k = 0; k < 3; ++k) {  // upper staples, nu descending
                const Mat3<float> t = mul_nn(lds_mat(cur + myop[3 * k] * SLOT_FLOATS), lds_mat(cur + myop[3 * k + 1] * SLOT_FLOATS));
                mac_na(acc, t, lds_mat(cur + myop[3 * k + 2] * SLOT_FLOATS));
                if (PLAQ && k == 2 - mu) plsum += (double)re_tr_na(lds_mat(cur + myop[18] * SLOT_FLOATS), acc);
            }
#pragma unroll 1
            for (int k = 3; k < 6; ++k) {  // lower staples, nu ascending
                const Mat3<float> t = mul_an(lds_mat(cur + myop[3 * k] * SLOT_FLOATS), lds_mat(cur + myop[3 * k + 1] * SLOT_FLOATS));
                mac_nn(acc, t, lds_mat(cur + myop[3 * k + 2] * SLOT_FLOATS));
            }
            const Mat3<float> umu = lds_mat(cur + myop[18] * SLOT_FLOATS);
            Mat3<float> r;
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = 0; b < 3; ++b) {
                    r.re[a][b] = fmaf(c1, acc.re[a][b], c0 * umu.re[a][b]);
                    r.im[a][b] = fmaf(c1, acc.im[a][b], c0 * umu.im[a][b]);
                }
            int org[4];
            tile_origin(tm, tile, org);
            const int s = (org[0] + lx[0]) + g.L[0] * ((org[1] + lx[1]) + g.L[1] * ((org[2] + lx[2]) + g.L[2] * (org[3] + lx[3])));
            store_mat(out.u[mu], s, r);
        }
        __syncthreads();  // the buffer just read is the target of the next iteration's copies
    }
    if (PLAQ) {
        double p[1] = {plsum};
        block_reduce_partial<1>(p, partials);
    }
}

}  // namespace

// --------------------------------------------------------------------------------------------
// host side: the two tables live in device memory per context until lqx_finalize
// --------------------------------------------------------------------------------------------
namespace {
struct DeviceTables {
    int nslots = 0;
    int* footprint = nullptr;
    unsigned short* operand = nullptr;
};
std::map<lqx_ctx*, DeviceTables> g_tables;
std::mutex g_tables_mutex;
}  // namespace

void lqx_staged_release(lqx_ctx* ctx) {
    std::lock_guard<std::mutex> lock(g_tables_mutex);
    auto it = g_tables.find(ctx);
    if (it == g_tables.end()) return;
    if (it->second.footprint) cudaFree(it->second.footprint);
    if (it->second.operand) cudaFree(it->second.operand);
    g_tables.erase(it);
}

// Returns LQX_OK, a negative status, or 1 if this lattice is not covered (extents must be multiples of 8x2x2x2).
int lqx_smear_staged_launch(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, double* plaq) {
    const Geo& g = ctx->geo;
    typedef Tiled<TX, TY, TZ, TT> MAP;
    if (!MAP::fits(g)) return 1;
    DeviceTables dt;
    {
        std::lock_guard<std::mutex> lock(g_tables_mutex);
        auto it = g_tables.find(ctx);
        if (it == g_tables.end()) {
            static const StagedTables host = build_tables();
            DeviceTables d;
            d.nslots = host.nslots;
            if (cudaMalloc(&d.footprint, host.footprint.size() * sizeof(int)) != cudaSuccess ||
                cudaMalloc(&d.operand, host.operand.size() * sizeof(unsigned short)) != cudaSuccess) {
                cudaGetLastError();
                if (d.footprint) cudaFree(d.footprint);
                return lqx_fail(ctx, LQX_ENOMEM, "staged smear tables");
            }
            LQX_CUDA(ctx, cudaMemcpyAsync(d.footprint, host.footprint.data(), host.footprint.size() * sizeof(int), cudaMemcpyHostToDevice, ctx->stream));
            LQX_CUDA(ctx, cudaMemcpyAsync(d.operand, host.operand.data(), host.operand.size() * sizeof(unsigned short), cudaMemcpyHostToDevice, ctx->stream));
            it = g_tables.insert(std::make_pair(ctx, d)).first;
        }
        dt = it->second;
    }
    const int ntiles = MAP::grid(g);
    const int nbuf = ctx->opt_tile == 2 ? 2 : 1;  // option "tile" = 2 selects the double-buffered one-CTA-per-SM form
    const int grid = std::min(ntiles, ctx->num_sms * (3 - nbuf));
    const TileMap tm = MAP::map(g, kSlabZ);
    const size_t smem = (size_t)nbuf * dt.nslots * SLOT_FLOATS * sizeof(float) + (size_t)dt.nslots * sizeof(int) + (size_t)NTHREADS * 19 * sizeof(unsigned short);
    if (plaq) {
        int rc = lqx_ensure_partials(ctx, (size_t)grid);
        if (rc) return rc;
    }
#define LQX_STAGED(P, NB)                                                                                                    \
    do {                                                                                                                     \
        LQX_CUDA(ctx, cudaFuncSetAttribute(k_smear_staged<P, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
        LqxTimed timed(ctx, LQX_K_SMEAR);                                                                                    \
        k_smear_staged<P, NB><<<grid, NTHREADS, smem, ctx->stream>>>(g, tm, in, out, c0, c1, ntiles, dt.nslots, dt.footprint, \
                                                                     dt.operand, plaq ? ctx->d_partials : nullptr);          \
    } while (0)
    if (plaq) {
        if (nbuf == 2) LQX_STAGED(true, 2); else LQX_STAGED(true, 1);
    } else {
        if (nbuf == 2) LQX_STAGED(false, 2); else LQX_STAGED(false, 1);
    }
#undef LQX_STAGED
    LQX_LAUNCH_CHECK(ctx);
    return plaq ? lqx_sum_partials(ctx, grid, 1, plaq) : LQX_OK;
}
