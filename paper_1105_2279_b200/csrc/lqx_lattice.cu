// lqx nearest-neighbour kernels: hop, plaquette (a8), and the C entry points of the
// staple sum / smear step (a7, kernels in lqx_smear.cu) and of the iterated smearing driver (a10).  Each is a single pass in which one thread
// evaluates the whole expression of its site, reading shifted operands at
// the periodic neighbour computed in-kernel (the role of the paper's site tables).
// CTAs own compact 4-d tiles (lqx_internal.cuh, Tiled<>) so that shared neighbours are L1 hits.
#include "lqx_internal.cuh"
#include "lqx_smear.cuh"

namespace {

// ---------------------------------------------------------------------------------------------
// hop: chi(x) = sum_mu U_mu(x) psi(x+mu^) + adj(U_mu(x-mu^)) psi(x-mu^)
// (Listing 1 lines 25/27 summed over mu; Eq. 2; BASELINE configs[1])
// ---------------------------------------------------------------------------------------------
template <typename T, int NSPIN, bool NORM2, typename MAP>
__global__ void __launch_bounds__(MAP::THREADS, (sizeof(T) == 4 ? 896 : 512) / MAP::THREADS) k_hop(const __grid_constant__ Geo g, const __grid_constant__ TileMap tm,
                                                      const __grid_constant__ Links<T> u, const T* __restrict__ psi, T* __restrict__ chi,
                                                      double* __restrict__ partials, unsigned int* ticket, double* __restrict__ out) {
    int x[4], s;
    double n2[1] = {0.0};
    if (MAP::site(g, tm, x, s)) {
        Vec3<T> acc[NSPIN];
#pragma unroll
        for (int a = 0; a < NSPIN; ++a)
#pragma unroll
            for (int i = 0; i < 3; ++i) acc[a].re[i] = acc[a].im[i] = T(0);
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            const int f = nbr_fwd(g, s, x, mu), b = nbr_bwd(g, s, x, mu);
            {
                const Mat3<T> m = load_mat(u.u[mu], s);
                Vec3<T> v[NSPIN];
                load_vecs<T, NSPIN>(psi, f, v);
#pragma unroll
                for (int a = 0; a < NSPIN; ++a) mac_mv(acc[a], m, v[a]);
            }
            {
                const Mat3<T> m = load_mat(u.u[mu], b);
                Vec3<T> v[NSPIN];
                load_vecs<T, NSPIN>(psi, b, v);
#pragma unroll
                for (int a = 0; a < NSPIN; ++a) mac_adj_mv(acc[a], m, v[a]);
            }
        }
        store_vecs<T, NSPIN>(chi, s, acc);
        if (NORM2) {
#pragma unroll
            for (int a = 0; a < NSPIN; ++a)
#pragma unroll
                for (int i = 0; i < 3; ++i) {
                    n2[0] = fma((double)acc[a].re[i], (double)acc[a].re[i], n2[0]);
                    n2[0] = fma((double)acc[a].im[i], (double)acc[a].im[i], n2[0]);
                }
        }
    }
    if (NORM2) block_reduce_finish<1>(n2, partials, ticket, out);
}

// ---------------------------------------------------------------------------------------------
// One iteration of the paper's Jacobi smearing routine (Listing 1 lines 20-30):
//   chi_new(x) = s_0(x) + kappa * sum_{mu != no_smear_dir} [U_mu(x) psi(x+mu^) + adj(U_mu(x-mu^)) psi(x-mu^)]
// i.e. E0 (psi = chi: here the ping-pong), E1, E2 x (Nd-1) and E3 of the listing in ONE pass instead of
// six; DIV: the last iteration also applies E4, chi /= norm (a true division, reading A22).
// dirmask bit mu = direction mu takes part.
// ---------------------------------------------------------------------------------------------
// Launch geometry (the paper's two tuning parameters): N_threads = blockDim.x (32..256)
// and N_site = NSITE sites per thread, taken grid-strided so that a warp still reads 32 consecutive sites.
// MASK >= 0: the set of smeared directions is a compile-time constant (all four, or all but time -- the two cases
// that occur), so the body is straight-line code and the loads of all directions can be in flight together;
// MASK < 0: the run-time dirmask decides per direction.
template <typename T, int NSPIN, bool DIV, int NSITE, int MASK>
__global__ void __launch_bounds__(256, sizeof(T) == 4 ? 3 : 2) k_jacobi_step(const __grid_constant__ Geo g, const __grid_constant__ Links<T> u,
                                                                             int dirmask, const T* __restrict__ psi, const T* __restrict__ s0,
                                                                             T kappa, T nrm, T* __restrict__ chi) {
    // Programmatic dependent launch (sm_90+): the iterations of the routine are launched with programmatic stream
    // serialisation, so the CTAs of iteration k+1 are scheduled -- and do their index arithmetic -- while iteration
    // k drains; they touch memory only after griddepcontrol.wait, which returns when iteration k is complete and
    // visible.  16^3x32, 20 iterations: 0.302 -> 0.268 ms.  (Requesting the first direction's links before the wait,
    // which do not depend on the previous iteration, changed nothing.)
    asm volatile("griddepcontrol.launch_dependents;");
    bool waited = false;
#pragma unroll 1
    for (int k = 0; k < NSITE; ++k) {
        const int s = (k * gridDim.x + blockIdx.x) * blockDim.x + threadIdx.x;
        if (s >= g.V) return;
        int x[4];
        site_coords(g, s, x);
        if (!waited) {
            asm volatile("griddepcontrol.wait;" ::: "memory");
            waited = true;
        }
        Vec3<T> acc[NSPIN];
#pragma unroll
        for (int a = 0; a < NSPIN; ++a)
#pragma unroll
            for (int i = 0; i < 3; ++i) acc[a].re[i] = acc[a].im[i] = T(0);
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            if (MASK >= 0 ? !((MASK >> mu) & 1) : !((dirmask >> mu) & 1)) continue;
            const int f = nbr_fwd(g, s, x, mu), b = nbr_bwd(g, s, x, mu);
            {
                const Mat3<T> m = load_mat(u.u[mu], s);
                Vec3<T> v[NSPIN];
                load_vecs<T, NSPIN>(psi, f, v);
#pragma unroll
                for (int a = 0; a < NSPIN; ++a) mac_mv(acc[a], m, v[a]);
            }
            {
                const Mat3<T> m = load_mat(u.u[mu], b);
                Vec3<T> v[NSPIN];
                load_vecs<T, NSPIN>(psi, b, v);
#pragma unroll
                for (int a = 0; a < NSPIN; ++a) mac_adj_mv(acc[a], m, v[a]);
            }
        }
        Vec3<T> src[NSPIN];
        load_vecs<T, NSPIN>(s0, s, src);
#pragma unroll
        for (int a = 0; a < NSPIN; ++a)
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                T re = fma(kappa, acc[a].re[i], src[a].re[i]), im = fma(kappa, acc[a].im[i], src[a].im[i]);
                if (DIV) {
                    re = re / nrm;
                    im = im / nrm;
                }
                acc[a].re[i] = re;
                acc[a].im[i] = im;
            }
        store_vecs<T, NSPIN>(chi, s, acc);
    }
}

// ---------------------------------------------------------------------------------------------
// plaquette: sum_{mu<nu} Re tr[U_mu(x) U_nu(x+mu^) adj(U_mu(x+nu^)) adj(U_nu(x))]
//          = sum_{mu<nu} Re tr[Q_munu(x) adj(Q_numu(x))],  Q_ab(x) = U_a(x) U_b(x+a^)
// ---------------------------------------------------------------------------------------------
template <typename T, typename MAP>
__global__ void __launch_bounds__(MAP::THREADS) k_plaquette(const __grid_constant__ Geo g, const __grid_constant__ TileMap tm,
                                                            const __grid_constant__ Links<T> u, double* __restrict__ partials) {
    int x[4], s;
    double p[1] = {0.0};
    if (MAP::site(g, tm, x, s)) {
        T acc = T(0);
#pragma unroll 1
        for (int mu = 0; mu < 3; ++mu) {
            const Mat3<T> a = load_mat(u.u[mu], s);
            const int xpmu = nbr_fwd(g, s, x, mu);
#pragma unroll 1
            for (int nu = mu + 1; nu < 4; ++nu) {
                const int xpnu = nbr_fwd(g, s, x, nu);
                const Mat3<T> q1 = mul_nn(a, load_mat(u.u[nu], xpmu));
                const Mat3<T> q2 = mul_nn(load_mat(u.u[nu], s), load_mat(u.u[mu], xpnu));
                acc += re_tr_na(q1, q2);
            }
        }
        p[0] = (double)acc;
    }
    block_reduce_partial<1>(p, partials);
}

// The same sum with the four links of the site held in registers and the plane loops unrolled: 16 instead of
// 21 matrix loads per site for about twice the registers (fp32: 165, three CTAs per SM).  The kernel is bound by
// the L1 data pipe rather than by latency -- spreading the six planes of a site over six warps (more loads in
// flight, 24 loads per site) ran 30-50 % slower -- so in fp32 the saved loads outweigh the lost occupancy
// (0.94 -> 0.86 ms at 48^3x96); in fp64 (254 registers) they do not (0.37 -> 0.39 ms at 32^3x64).
template <typename T, int MINB>
__global__ void __launch_bounds__(128, MINB) k_plaquette_held(const __grid_constant__ Geo g, const __grid_constant__ Links<T> u,
                                                              double* __restrict__ partials) {
    const int s = blockIdx.x * 128 + threadIdx.x;
    double p[1] = {0.0};
    if (s < g.V) {
        int x[4];
        site_coords(g, s, x);
        Mat3<T> own[4];
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) own[mu] = load_mat(u.u[mu], s);
        T acc = T(0);
#pragma unroll
        for (int mu = 0; mu < 3; ++mu) {
            const int xpmu = nbr_fwd(g, s, x, mu);
#pragma unroll
            for (int nu = mu + 1; nu < 4; ++nu) {
                const int xpnu = nbr_fwd(g, s, x, nu);
                const Mat3<T> q1 = mul_nn(own[mu], load_mat(u.u[nu], xpmu));
                const Mat3<T> q2 = mul_nn(own[nu], load_mat(u.u[mu], xpnu));
                acc += re_tr_na(q1, q2);
            }
        }
        p[0] = (double)acc;
    }
    block_reduce_partial<1>(p, partials);
}

int check_links(lqx_ctx** ctx_out, const lqx_field* const u[4]) {
    if (!u) return LQX_EINVAL;
    lqx_ctx* ctx = nullptr;
    for (int mu = 0; mu < 4; ++mu) {
        if (!u[mu]) return LQX_EINVAL;
        if (!ctx) ctx = u[mu]->ctx;
        if (u[mu]->ctx != ctx) return lqx_fail(ctx, LQX_EGEOM, "links belong to different contexts");
        if (u[mu]->kind != LQX_COLORMAT) return lqx_fail(ctx, LQX_ETYPE, "links must be colour matrices");
        if (u[mu]->prec != u[0]->prec) return lqx_fail(ctx, LQX_ETYPE, "mixed precision links");
    }
    *ctx_out = ctx;
    return LQX_OK;
}


template <typename T>
int plaquette_launch(lqx_ctx* ctx, const lqx_field* const u[4], double* out) {
    const Geo& g = ctx->geo;
    const int choice = lqx_pick_tile(ctx, 0);  // measured: linear 128-site blocks beat every tile shape here
    int nblocks = 0;
    // option plaq_variant: 0 = automatic (held links in fp32, rolled loops in fp64: measured), 1 = rolled, 2 = held
    const int pv = ctx->opt_plaq_variant ? ctx->opt_plaq_variant : ctx->tuned_plaq_variant[sizeof(T) == 4 ? 0 : 1];
    const bool held = pv == 2 || (pv == 0 && sizeof(T) == 4 && choice == 0);
    if (held) {
        nblocks = (g.V + 127) / 128;
        int rc = lqx_ensure_partials(ctx, (size_t)nblocks);
        if (rc) return rc;
        {
            LqxTimed timed(ctx, LQX_K_PLAQUETTE);
            k_plaquette_held<T, sizeof(T) == 4 ? 3 : 1><<<nblocks, 128, 0, ctx->stream>>>(g, make_links<T>(u), ctx->d_partials);
        }
        LQX_LAUNCH_CHECK(ctx);
        return lqx_sum_partials(ctx, nblocks, 1, out);
    }
    LQX_WITH_MAP(choice, {
        const int grid = MAP::grid(g);
        nblocks = grid;
        int rc = lqx_ensure_partials(ctx, (size_t)grid);
        if (rc) return rc;
        LqxTimed timed(ctx, LQX_K_PLAQUETTE);
        k_plaquette<T, MAP><<<grid, MAP::THREADS, 0, ctx->stream>>>(g, MAP::map(g, kSlabZ), make_links<T>(u), ctx->d_partials);
    })
    LQX_LAUNCH_CHECK(ctx);
    return lqx_sum_partials(ctx, nblocks, 1, out);
}

// the plaquette sum over the sites of the time slices [t0, t1) only (NEXT-4: a rank's own slab)
template <typename T>
int plaquette_range_launch(lqx_ctx* ctx, const lqx_field* const u[4], int t0, int t1, double* out) {
    const Geo& g = ctx->geo;
    TileMap tm = Linear::map(g, kSlabZ);
    const int grid = Linear::restrict_t(g, tm, t0, t1);
    int rc = lqx_ensure_partials(ctx, (size_t)grid);
    if (rc) return rc;
    {
        LqxTimed timed(ctx, LQX_K_PLAQUETTE);
        k_plaquette<T, Linear><<<grid, Linear::THREADS, 0, ctx->stream>>>(g, tm, make_links<T>(u), ctx->d_partials);
    }
    LQX_LAUNCH_CHECK(ctx);
    return lqx_sum_partials(ctx, grid, 1, out);
}

}  // namespace

int lqx_pick_tile(const lqx_ctx* ctx, int first_choice) {
    const Geo& g = ctx->geo;
    auto fits = [&](int c) {
        switch (c) {
            case 0: return true;
            case 1: return TileA::fits(g);
            case 2: return TileB::fits(g);
            case 3: return TileC::fits(g);
            case 4: return TileD::fits(g);
            case 5: return TileE::fits(g);
            case 6: return TileF::fits(g);
            default: return false;
        }
    };
    if (ctx->opt_tile >= 0 && fits(ctx->opt_tile)) return ctx->opt_tile;
    if (fits(first_choice)) return first_choice;
    static const int order[kNumTiles] = {4, 1, 5, 2, 3, 6};
    for (int c : order)
        if (fits(c)) return c;
    return 0;
}

// =============================================================================================
// C entry points
// =============================================================================================
static int hop_impl(lqx_field* chi, const lqx_field* const u[4], const lqx_field* psi, double* norm2_out) {
    lqx_ctx* ctx;
    int rc = check_links(&ctx, u);
    if (rc) return rc;
    if (!chi || !psi) return LQX_EINVAL;
    if (chi->ctx != ctx || psi->ctx != ctx) return lqx_fail(ctx, LQX_EGEOM, "hop: different contexts");
    if (chi->prec != u[0]->prec || psi->prec != u[0]->prec) return lqx_fail(ctx, LQX_ETYPE, "hop: mixed precision");
    if (chi->kind != psi->kind || (psi->kind != LQX_FERMION && psi->kind != LQX_COLORVEC))
        return lqx_fail(ctx, LQX_ETYPE, "hop: psi/chi must both be fermions or colour vectors");
    if (lqx_same(chi, psi)) return lqx_fail(ctx, LQX_EALIAS, "hop: chi aliases psi");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const Geo& g = ctx->geo;
    const bool n2 = norm2_out != nullptr;
    const bool ferm = psi->kind == LQX_FERMION;
    const int choice = lqx_pick_tile(ctx, 0);  // measured: linear blocks beat every tile shape for the hop
#define LQX_HOP(T, NSPIN, N2)                                                                                      \
    k_hop<T, NSPIN, N2, MAP><<<grid, MAP::THREADS, 0, ctx->stream>>>(g, tm, make_links<T>(u), (const T*)psi->data, \
                                                                    (T*)chi->data, ctx->d_partials, ctx->d_ticket, ctx->h_result)
#define LQX_HOP_BODY                                                                                  \
    {                                                                                                 \
        const int grid = MAP::grid(g);                                                                \
        if (n2) {                                                                                     \
            rc = lqx_ensure_partials(ctx, (size_t)grid);                                              \
            if (rc) return rc;                                                                        \
        }                                                                                             \
        const TileMap tm = MAP::map(g, kSlabZ);                                                       \
        LqxTimed timed(ctx, LQX_K_HOP);                                                               \
        if (psi->prec == LQX_F32) {                                                                   \
            if (ferm) { if (n2) LQX_HOP(float, 4, true); else LQX_HOP(float, 4, false); }             \
            else      { if (n2) LQX_HOP(float, 1, true); else LQX_HOP(float, 1, false); }             \
        } else {                                                                                      \
            if (ferm) { if (n2) LQX_HOP(double, 4, true); else LQX_HOP(double, 4, false); }           \
            else      { if (n2) LQX_HOP(double, 1, true); else LQX_HOP(double, 1, false); }           \
        }                                                                                             \
    }
    // linear blocks: the CTA size is a launch-geometry knob (option "hop_block", the auto-tuner's choice)
    const int hb = ctx->opt_hop_block ? ctx->opt_hop_block : ctx->tuned_hop_block[psi->prec == LQX_F32 ? 0 : 1];
    if (choice == 0 && hb == 32) { typedef LinearN<32> MAP; LQX_HOP_BODY }
    else if (choice == 0 && hb == 64) { typedef LinearN<64> MAP; LQX_HOP_BODY }
    else if (choice == 0 && hb == 256) { typedef LinearN<256> MAP; LQX_HOP_BODY }
    else LQX_WITH_MAP(choice, LQX_HOP_BODY)
#undef LQX_HOP_BODY
#undef LQX_HOP
    LQX_LAUNCH_CHECK(ctx);
    if (n2) return lqx_fetch_result(ctx, 1, norm2_out);
    return LQX_OK;
}

extern "C" int lqx_hop(lqx_field* chi, const lqx_field* const u[4], const lqx_field* psi) {
    return hop_impl(chi, u, psi, nullptr);
}
extern "C" int lqx_hop_norm2(lqx_field* chi, const lqx_field* const u[4], const lqx_field* psi, double* norm2_out) {
    if (!norm2_out) return LQX_EINVAL;
    return hop_impl(chi, u, psi, norm2_out);
}

extern "C" int lqx_plaquette(const lqx_field* const u[4], double* plaq_sum, double* plaq_avg) {
    lqx_ctx* ctx;
    int rc = check_links(&ctx, u);
    if (rc) return rc;
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    rc = u[0]->prec == LQX_F32 ? plaquette_launch<float>(ctx, u, ctx->h_result) : plaquette_launch<double>(ctx, u, ctx->h_result);
    if (rc) return rc;
    double p;
    rc = lqx_fetch_result(ctx, 1, &p);
    if (rc) return rc;
    if (plaq_sum) *plaq_sum = p;
    if (plaq_avg) *plaq_avg = p / (18.0 * (double)ctx->geo.V);
    return LQX_OK;
}

extern "C" int lqx_plaquette_range(const lqx_field* const u[4], int t0, int t1, double* plaq_sum) {
    lqx_ctx* ctx;
    int rc = check_links(&ctx, u);
    if (rc) return rc;
    if (!plaq_sum) return LQX_EINVAL;
    if (t0 < 0 || t1 > ctx->geo.L[3] || t0 >= t1) return lqx_fail(ctx, LQX_EINVAL, "plaquette_range: 0 <= t0 < t1 <= L3");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    rc = u[0]->prec == LQX_F32 ? plaquette_range_launch<float>(ctx, u, t0, t1, ctx->h_result)
                               : plaquette_range_launch<double>(ctx, u, t0, t1, ctx->h_result);
    if (rc) return rc;
    return lqx_fetch_result(ctx, 1, plaq_sum);
}

extern "C" int lqx_field_slice(const lqx_field* f, int t, int64_t* offset_bytes, int64_t* nbytes) {
    if (!f || !offset_bytes || !nbytes) return LQX_EINVAL;
    lqx_ctx* ctx = f->ctx;
    const Geo& g = ctx->geo;
    const int64_t v3 = (int64_t)g.L[0] * g.L[1] * g.L[2];
    if (t < 0 || t >= g.L[3]) return lqx_fail(ctx, LQX_EINVAL, "field_slice: t out of range");
    if (v3 % 32 != 0) return lqx_fail(ctx, LQX_EGEOM, "field_slice: a time slice is contiguous only if L0*L1*L2 is a multiple of 32");
    const int64_t per_site = 2 * (int64_t)(int)f->kind * (int64_t)(int)f->prec;
    *offset_bytes = (int64_t)t * v3 * per_site;
    *nbytes = v3 * per_site;
    return LQX_OK;
}

static int check_smear_args(lqx_ctx** ctx_out, lqx_field* const uout[4], const lqx_field* const uin[4]) {
    lqx_ctx* ctx;
    int rc = check_links(&ctx, uin);
    if (rc) return rc;
    rc = check_links(&ctx, (const lqx_field* const*)uout);
    if (rc) return rc;
    if (uout[0]->ctx != uin[0]->ctx) return lqx_fail(ctx, LQX_EGEOM, "smear: different contexts");
    if (uout[0]->prec != uin[0]->prec) return lqx_fail(ctx, LQX_ETYPE, "smear: mixed precision");
    for (int a = 0; a < 4; ++a)
        for (int b = 0; b < 4; ++b) {
            if (lqx_same(uout[a], uin[b])) return lqx_fail(ctx, LQX_EALIAS, "smear: output aliases an input link field");
            if (a != b && lqx_same(uout[a], uout[b])) return lqx_fail(ctx, LQX_EALIAS, "smear: outputs alias each other");
        }
    *ctx_out = ctx;
    return LQX_OK;
}

extern "C" int lqx_staple_sum(lqx_field* out, const lqx_field* const u[4], int mu) {
    lqx_ctx* ctx;
    int rc = check_links(&ctx, u);
    if (rc) return rc;
    if (!out) return LQX_EINVAL;
    if (mu < 0 || mu > 3) return lqx_fail(ctx, LQX_EINVAL, "mu");
    if (out->ctx != ctx) return lqx_fail(ctx, LQX_EGEOM, "staple_sum: different contexts");
    if (out->kind != LQX_COLORMAT || out->prec != u[0]->prec) return lqx_fail(ctx, LQX_ETYPE, "staple_sum: output type");
    for (int b = 0; b < 4; ++b)
        if (lqx_same(out, u[b])) return lqx_fail(ctx, LQX_EALIAS, "staple_sum: output aliases a link field");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    lqx_field* o[4] = {out, nullptr, nullptr, nullptr};
    return lqx_smear_launch(ctx, o, u, 0.0, mu, nullptr);
}

extern "C" int lqx_smear_step(lqx_field* const uout[4], const lqx_field* const uin[4], double alpha,
                              double* plaq_in_or_null) {
    if (!uout || !uin) return LQX_EINVAL;
    lqx_ctx* ctx;
    int rc = check_smear_args(&ctx, uout, uin);
    if (rc) return rc;
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    rc = lqx_smear_launch(ctx, uout, uin, alpha, -1, plaq_in_or_null ? ctx->h_result : nullptr);
    if (rc) return rc;
    if (plaq_in_or_null) return lqx_fetch_result(ctx, 1, plaq_in_or_null);
    return LQX_OK;
}

// NEXT-4 building block: the smear step of the time slices [t0, t1) only.  Asynchronous; the caller guarantees that the
// input slices t0-1 .. t1 (periodic in the context's t extent) hold what the step should read -- on a t-slab with halo
// slices that is "after the halo exchange".  Same per-site arithmetic as lqx_smear_step, bit for bit.
extern "C" int lqx_smear_step_range(lqx_field* const uout[4], const lqx_field* const uin[4], double alpha, int t0, int t1) {
    if (!uout || !uin) return LQX_EINVAL;
    lqx_ctx* ctx;
    int rc = check_smear_args(&ctx, uout, uin);
    if (rc) return rc;
    if (t0 < 0 || t1 > ctx->geo.L[3] || t0 >= t1) return lqx_fail(ctx, LQX_EINVAL, "smear_step_range: 0 <= t0 < t1 <= L3");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    rc = lqx_smear_launch_range_any(ctx, uout, uin, alpha, t0, t1);
    return rc == 1 ? lqx_fail(ctx, LQX_EGEOM, "smear_step_range: no kernel map splits at these time slices") : rc;
}

extern "C" int lqx_smear_iterate(lqx_field* const u[4], lqx_field* const tmp[4], double alpha, int nsteps,
                                 double* plaq_avg_after_each) {
    if (!u || !tmp) return LQX_EINVAL;
    lqx_ctx* ctx;
    int rc = check_smear_args(&ctx, tmp, (const lqx_field* const*)u);
    if (rc) return rc;
    if (nsteps < 0) return lqx_fail(ctx, LQX_EINVAL, "nsteps < 0");
    if (nsteps == 0) return LQX_OK;
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    // per-step plaquette sums: the kernels write them straight into pinned host memory
    const bool want = plaq_avg_after_each != nullptr;
    double* res = nullptr;
    bool res_owned = false;
    if (want) {
        if (nsteps <= 64) {
            res = ctx->h_result;
        } else {
            if (cudaHostAlloc(&res, (size_t)nsteps * sizeof(double), cudaHostAllocPortable | cudaHostAllocMapped) != cudaSuccess) {
                cudaGetLastError();
                return lqx_fail(ctx, LQX_ENOMEM, "plaquette results");
            }
            res_owned = true;
        }
    }
    // Ping-pong u -> tmp -> u ...  The plaquette of the field after step k is the plaquette of the
    // INPUT of step k+1, which that step's kernel accumulates for free; only the last one needs its
    // own pass.
    lqx_field* const* src = u;
    lqx_field* const* dst = tmp;
    for (int k = 0; k < nsteps && rc == LQX_OK; ++k) {
        double* dp = (want && k > 0) ? res + (k - 1) : nullptr;
        rc = lqx_smear_launch(ctx, dst, (const lqx_field* const*)src, alpha, -1, dp);
        std::swap(src, dst);
    }
    // result is in src now; if that is tmp (odd nsteps), copy back into u
    if (rc == LQX_OK && src != u) {
        for (int mu = 0; mu < 4 && rc == LQX_OK; ++mu) rc = lqx_copy(u[mu], tmp[mu]);
    }
    if (rc == LQX_OK && want) {
        rc = u[0]->prec == LQX_F32 ? plaquette_launch<float>(ctx, (const lqx_field* const*)u, res + (nsteps - 1))
                                   : plaquette_launch<double>(ctx, (const lqx_field* const*)u, res + (nsteps - 1));
    }
    if (rc == LQX_OK) {
        cudaError_t e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) rc = lqx_cuda_fail(ctx, e, "smear_iterate sync");
    }
    if (rc == LQX_OK && want) {
        const double norm = 18.0 * (double)ctx->geo.V;
        for (int k = 0; k < nsteps; ++k) plaq_avg_after_each[k] = res[k] / norm;
    }
    if (res_owned) cudaFreeHost(res);
    return rc;
}

// Streamed one-step host path: the lattice is cut into slabs of time slices; slab k is uploaded (and converted to the
// blocked layout on the context's stream) on an upload stream, smeared on the context's stream as soon as its two
// neighbour slabs are in, converted back and downloaded on a download stream -- so the PCIe link carries both directions at once and the
// kernels hide under the copies.  A slab is a contiguous site range in QDP order and in the blocked layout alike
// (t is the slowest index), provided its volume is a multiple of the 32-site block.
// Returns the slab thickness (time slices) to use, or 0 if this lattice / option setting does not stream.
static int host_slab_thickness(const lqx_ctx* ctx, lqx_prec prec) {
    const Geo& g = ctx->geo;
    if (ctx->opt_host_slabs == 0) return 0;
    if (ctx->opt_smear_variant != 0 && ctx->opt_smear_variant != 3 && ctx->opt_smear_variant != 9 && ctx->opt_smear_variant != 10) return 0;  // only the literal kernels take a t-range
    // automatic: at most 48 slabs (the three slabs left after the last upload are the un-overlapped tail: 48 slabs at
    // configs[3] measured 68-71 ms per call, 24: 72-75, 12: 76-78, serial: 119) of at least 4 MB per link, below
    // which the per-slab launches and copies cost more than the overlap gains; option "host_slabs" = n > 0 forces
    // up to n slabs whatever their size
    const bool forced = ctx->opt_host_slabs > 0;
    const int max_slabs = forced ? ctx->opt_host_slabs : 48;
    const int64_t min_bytes = forced ? 0 : (int64_t)4 << 20;
    const int64_t v3 = (int64_t)g.L[0] * g.L[1] * g.L[2];
    for (int th = 2; th * 3 <= g.L[3]; th += 2) {  // even: every tile shape has a t-extent of 1 or 2
        if (g.L[3] % th || (v3 * th) % 32) continue;
        if (g.L[3] / th <= max_slabs && v3 * th * 18 * (int)prec >= min_bytes) return th;
    }
    return 0;
}

static int smear_host_streamed(lqx_ctx* ctx, lqx_prec prec, const void* const host_u_in[4], void* const host_u_out[4],
                               double alpha, int th, double* plaq_avg) {
    const Geo& g = ctx->geo;
    const int K = g.L[3] / th;
    int rc = LQX_OK;
    for (int k = 8; k < 12 && rc == LQX_OK; ++k)
        if (!ctx->host_work[k]) rc = lqx_field_alloc(ctx, LQX_COLORMAT, prec, &ctx->host_work[k]);
    if (rc != LQX_OK) return rc;
    for (int k = 0; k < 2; ++k)
        if (!ctx->pipe_stream[k]) LQX_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->pipe_stream[k], cudaStreamNonBlocking));
    while ((int)ctx->pipe_events.size() < 2 * K + 2) {
        cudaEvent_t e;
        LQX_CUDA(ctx, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        ctx->pipe_events.push_back(e);
    }
    lqx_field* const* u = ctx->host_work;       // input links, blocked layout
    lqx_field* const* t = ctx->host_work + 4;   // smeared links, blocked layout
    lqx_field* const* q = ctx->host_work + 8;   // QDP-order staging: slab k holds the input until it is converted,
                                                // then the output from its conversion until it is downloaded
    cudaStream_t up = ctx->pipe_stream[0], down = ctx->pipe_stream[1], main = ctx->stream;
    cudaEvent_t* ev_in = ctx->pipe_events.data();        // [K]  slab uploaded
    cudaEvent_t* ev_out = ctx->pipe_events.data() + K;   // [K]  slab smeared and converted back
    cudaEvent_t ev_begin = ctx->pipe_events[2 * K], ev_end = ctx->pipe_events[2 * K + 1];
    const size_t slab_sites = (size_t)g.L[0] * g.L[1] * g.L[2] * th;
    const size_t slab_bytes = slab_sites * 18 * (int)prec;
    const int slab_blocks = (int)(slab_sites / 32);
    // a failing runtime call records the error in rc and the remaining steps are skipped; the join below still runs
#define PIPE_TRY(call)                                                                       \
    do {                                                                                     \
        if (rc == LQX_OK) {                                                                  \
            cudaError_t e__ = (call);                                                        \
            if (e__ != cudaSuccess) rc = lqx_cuda_fail(ctx, e__, #call);                     \
        }                                                                                    \
    } while (0)
    // everything enqueued earlier on the context's stream comes first
    PIPE_TRY(cudaEventRecord(ev_begin, main));
    PIPE_TRY(cudaStreamWaitEvent(up, ev_begin, 0));
    PIPE_TRY(cudaStreamWaitEvent(down, ev_begin, 0));
    auto smear_slab = [&](int j) -> int {
        int r = lqx_smear_launch_range(ctx, t, (const lqx_field* const*)u, alpha, j * th, (j + 1) * th);
        if (r > 0) r = lqx_fail(ctx, LQX_EGEOM, "smear_iterate_host: tile does not split at the slab boundary");
        for (int mu = 0; mu < 4 && r == LQX_OK; ++mu)
            r = lqx_transpose_range(ctx, LQX_COLORMAT, prec, t[mu]->data, q[mu]->data, false, j * slab_blocks, slab_blocks, main);
        if (r != LQX_OK) return r;
        PIPE_TRY(cudaEventRecord(ev_out[j], main));
        PIPE_TRY(cudaStreamWaitEvent(down, ev_out[j], 0));
        for (int mu = 0; mu < 4 && rc == LQX_OK; ++mu)
            PIPE_TRY(cudaMemcpyAsync((char*)host_u_out[mu] + (size_t)j * slab_bytes, (const char*)q[mu]->data + (size_t)j * slab_bytes,
                                          slab_bytes, cudaMemcpyDeviceToHost, down));
        return rc;
    };
    for (int k = 0; k < K && rc == LQX_OK; ++k) {
        for (int mu = 0; mu < 4 && rc == LQX_OK; ++mu)
            PIPE_TRY(cudaMemcpyAsync((char*)q[mu]->data + (size_t)k * slab_bytes, (const char*)host_u_in[mu] + (size_t)k * slab_bytes,
                                          slab_bytes, cudaMemcpyHostToDevice, up));
        // the side streams carry copies only, so neither copy engine ever waits for a kernel
        PIPE_TRY(cudaEventRecord(ev_in[k], up));
        PIPE_TRY(cudaStreamWaitEvent(main, ev_in[k], 0));
        for (int mu = 0; mu < 4 && rc == LQX_OK; ++mu)
            rc = lqx_transpose_range(ctx, LQX_COLORMAT, prec, q[mu]->data, u[mu]->data, true, k * slab_blocks, slab_blocks, main);
        if (rc != LQX_OK) break;
        // slab k-1 has both neighbours now (slabs 0 and K-1 wait for the wrap-around, below)
        if (k >= 2) rc = smear_slab(k - 1);
    }
    if (rc == LQX_OK) rc = smear_slab(K - 1);
    if (rc == LQX_OK) rc = smear_slab(0);
    if (rc == LQX_OK && plaq_avg)
        rc = prec == LQX_F32 ? plaquette_launch<float>(ctx, (const lqx_field* const*)t, ctx->h_result)
                             : plaquette_launch<double>(ctx, (const lqx_field* const*)t, ctx->h_result);
#undef PIPE_TRY
    // join the side streams into the context's stream even on failure, so nothing is left in flight
    cudaEventRecord(ev_end, down);
    cudaStreamWaitEvent(main, ev_end, 0);
    cudaEventRecord(ev_end, up);
    cudaStreamWaitEvent(main, ev_end, 0);
    cudaError_t e = cudaStreamSynchronize(main);
    if (rc == LQX_OK && e != cudaSuccess) rc = lqx_cuda_fail(ctx, e, "smear_iterate_host sync");
    if (rc == LQX_OK && plaq_avg) plaq_avg[0] = ctx->h_result[0] / (18.0 * (double)g.V);
    return rc;
}

extern "C" int lqx_smear_iterate_host(lqx_ctx* ctx, lqx_prec prec, const void* const host_u_in[4],
                                      void* const host_u_out[4], double alpha, int nsteps,
                                      double* plaq_avg_after_each) {
    if (!ctx || !host_u_in || !host_u_out) return LQX_EINVAL;
    for (int mu = 0; mu < 4; ++mu)
        if (!host_u_in[mu] || !host_u_out[mu]) return LQX_EINVAL;
    if (prec != LQX_F32 && prec != LQX_F64) return LQX_EINVAL;
    int rc = LQX_OK;
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    // the work fields (links + ping-pong scratch + staging) are kept in the context between calls: allocating and
    // freeing 6 GB per call costs more than the transfers (and varies wildly); lqx_finalize releases them
    if (ctx->host_work[0] && ctx->host_work[0]->prec != prec) {
        LQX_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        for (int k = 0; k < 12; ++k) {
            if (ctx->host_work[k]) lqx_field_free(ctx->host_work[k]);
            ctx->host_work[k] = nullptr;
        }
    }
    for (int k = 0; k < 8 && rc == LQX_OK; ++k)
        if (!ctx->host_work[k]) rc = lqx_field_alloc(ctx, LQX_COLORMAT, prec, &ctx->host_work[k]);
    if (rc != LQX_OK) return rc;
    if (nsteps == 1) {
        const int th = host_slab_thickness(ctx, prec);
        if (th > 0) return smear_host_streamed(ctx, prec, host_u_in, host_u_out, alpha, th, plaq_avg_after_each);
    }
    lqx_field* const* u = ctx->host_work;
    lqx_field* const* t = ctx->host_work + 4;
    // all four uploads and conversions are enqueued back to back (no host round trip between them); the
    // smear kernels follow in stream order; the four downloads are enqueued likewise and ONE synchronisation
    // ends the call, after which the host buffers are no longer touched
    for (int mu = 0; mu < 4 && rc == LQX_OK; ++mu) rc = lqx_push_impl(u[mu], host_u_in[mu], false);
    if (rc == LQX_OK) rc = lqx_smear_iterate(u, t, alpha, nsteps, plaq_avg_after_each);
    for (int mu = 0; mu < 4 && rc == LQX_OK; ++mu) rc = lqx_pop_impl(u[mu], host_u_out[mu], false);
    {
        cudaError_t e = cudaStreamSynchronize(ctx->stream);
        if (rc == LQX_OK && e != cudaSuccess) rc = lqx_cuda_fail(ctx, e, "smear_iterate_host sync");
    }
    return rc;
}

// The paper's routine (Listing 1): chi <- sum_{n<=iter} kappa^n H^n chi / norm.
extern "C" int lqx_jacobi_smear(lqx_field* chi, const lqx_field* const u[4], double kappa, int iter, int no_smear_dir,
                                double norm, lqx_field* const tmp[2]) {
    lqx_ctx* ctx;
    int rc = check_links(&ctx, u);
    if (rc) return rc;
    if (!chi || !tmp || !tmp[0] || !tmp[1]) return LQX_EINVAL;
    if (iter < 0) return lqx_fail(ctx, LQX_EINVAL, "jacobi_smear: iter < 0");
    if (norm == 0.0) return lqx_fail(ctx, LQX_EINVAL, "jacobi_smear: norm == 0");
    if (chi->kind != LQX_FERMION && chi->kind != LQX_COLORVEC) return lqx_fail(ctx, LQX_ETYPE, "jacobi_smear: chi must be a fermion or a colour vector");
    for (int k = 0; k < 2; ++k) {
        if (tmp[k]->ctx != ctx || chi->ctx != ctx) return lqx_fail(ctx, LQX_EGEOM, "jacobi_smear: different contexts");
        if (tmp[k]->kind != chi->kind || tmp[k]->prec != chi->prec) return lqx_fail(ctx, LQX_ETYPE, "jacobi_smear: scratch fields must match chi");
        if (lqx_same(tmp[k], chi)) return lqx_fail(ctx, LQX_EALIAS, "jacobi_smear: scratch aliases chi");
    }
    if (lqx_same(tmp[0], tmp[1])) return lqx_fail(ctx, LQX_EALIAS, "jacobi_smear: scratch fields alias each other");
    if (chi->prec != u[0]->prec) return lqx_fail(ctx, LQX_ETYPE, "jacobi_smear: mixed precision");
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    if (iter == 0) return lqx_divide(chi, chi, norm);  // s_0 = chi; chi /= norm
    const Geo& g = ctx->geo;
    int dirmask = 0xF;
    if (no_smear_dir >= 0 && no_smear_dir < 4) dirmask &= ~(1 << no_smear_dir);
    // s_0 = chi (E0, Listing line 16).  The iterate ping-pongs so that the last write lands in chi: for an odd
    // iteration count the first iteration reads the copy and writes chi, otherwise it reads chi and writes tmp[1].
    rc = lqx_copy(tmp[0], chi);
    if (rc) return rc;
    const lqx_field* cur = (iter & 1) ? tmp[0] : chi;
    lqx_field* nxt = (iter & 1) ? chi : tmp[1];
    // launch geometry: options "jacobi_block" (N_threads: 32, 64, 128, 256) and "jacobi_sites" (N_site: 1, 2, 4)
    // defaults from the sweep on B200 (bench.py --sweep-geometry): 32 x 1 in fp32 -- as on the
    // paper's GTX 480 --, 128 x 1 in fp64 (where the block size makes no measurable difference)
    const int pi = chi->prec == LQX_F32 ? 0 : 1;
    const int ob = ctx->opt_jacobi_block ? ctx->opt_jacobi_block : ctx->tuned_jacobi_block[pi];
    const int os = ctx->opt_jacobi_sites ? ctx->opt_jacobi_sites : ctx->tuned_jacobi_sites[pi];
    const int bs = (ob == 32 || ob == 64 || ob == 128 || ob == 256) ? ob : (chi->prec == LQX_F32 ? 32 : 128);
    const int nsite = (os == 2 || os == 4) ? os : 1;
    const int grid = (g.V + bs * nsite - 1) / (bs * nsite);
    const bool ferm = chi->kind == LQX_FERMION;
    for (int it = 0; it < iter; ++it) {
        const bool last = it == iter - 1;
        {
            LqxTimed timed(ctx, LQX_K_HOP);
#define LQX_JAC3(T, NSPIN, DIV, NS, MASK)                                                                                  \
    do {                                                                                                                   \
        cudaLaunchConfig_t cfg = {};                                                                                       \
        cfg.gridDim = dim3(grid), cfg.blockDim = dim3(bs), cfg.dynamicSmemBytes = 0, cfg.stream = ctx->stream;             \
        cudaLaunchAttribute attr[1];                                                                                       \
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;                                                   \
        attr[0].val.programmaticStreamSerializationAllowed = 1;                                                            \
        cfg.attrs = attr, cfg.numAttrs = 1;                                                                                \
        LQX_CUDA(ctx, cudaLaunchKernelEx(&cfg, k_jacobi_step<T, NSPIN, DIV, NS, MASK>, g, make_links<T>(u), dirmask,       \
                                         (const T*)cur->data, (const T*)tmp[0]->data, (T)kappa, (T)norm, (T*)nxt->data)); \
    } while (0)
#define LQX_JAC(T, NSPIN, DIV)                                          \
    do {                                                                \
        if (nsite == 1 && dirmask == 0xF) LQX_JAC3(T, NSPIN, DIV, 1, 0xF); \
        else if (nsite == 1 && dirmask == 0x7) LQX_JAC3(T, NSPIN, DIV, 1, 0x7); \
        else if (nsite == 1) LQX_JAC3(T, NSPIN, DIV, 1, -1);            \
        else if (nsite == 2) LQX_JAC3(T, NSPIN, DIV, 2, -1);            \
        else LQX_JAC3(T, NSPIN, DIV, 4, -1);                            \
    } while (0)
            if (chi->prec == LQX_F32) {
                if (ferm) { if (last) LQX_JAC(float, 4, true); else LQX_JAC(float, 4, false); }
                else      { if (last) LQX_JAC(float, 1, true); else LQX_JAC(float, 1, false); }
            } else {
                if (ferm) { if (last) LQX_JAC(double, 4, true); else LQX_JAC(double, 4, false); }
                else      { if (last) LQX_JAC(double, 1, true); else LQX_JAC(double, 1, false); }
            }
#undef LQX_JAC
#undef LQX_JAC3
        }
        LQX_LAUNCH_CHECK(ctx);
        cur = nxt;
        nxt = (nxt == chi) ? tmp[1] : chi;
    }
    return LQX_OK;
}
