// lqx_autotune: the paper's "auto-tuning of the geometry parameters ... stored for later inclusion" (PAPER.md:128
// sec.5.4; to-do list, sec.9; the sweeps it would automate: sec.8, Figs. 1-2).
//
// For one kernel class and precision the tuner times every launch geometry the library can select -- CTA size,
// sites per thread, CTA tile shape, kernel variant -- on the CONTEXT'S OWN lattice, with CUDA events on the context's
// stream, and keeps the fastest in the context: later calls of that class use it unless an explicit option overrides it.
// Every candidate is a geometry the parity tests run against the oracle (tests/test_gpu_parity.py: smear variants and
// tiles, plaquette variants, hop block sizes, Jacobi N_threads x N_site).  The timings are returned as a table
// (bench.py prints it: the B200 counterpart of the paper's Figs. 1-2).
#include <algorithm>
#include <vector>

#include "lqx_internal.cuh"
#include "lqx_smear.cuh"

namespace {

struct Scratch {  // fields of the tuning run; freed on every exit path
    std::vector<lqx_field*> f;
    ~Scratch() {
        for (lqx_field* p : f) lqx_field_free(p);
    }
    lqx_field* get(lqx_ctx* ctx, lqx_kind k, lqx_prec p) {
        lqx_field* h = nullptr;
        if (lqx_field_alloc(ctx, k, p, &h) != LQX_OK) return nullptr;
        f.push_back(h);
        return h;
    }
};

// unit links / a constant vector: timing does not depend on the values, only NaNs and denormals must be avoided
template <typename T>
__global__ void k_fill_unit(int V, int nreal, T* __restrict__ dst, int diag_stride) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= V) return;
    for (int r = 0; r < nreal; ++r) {
        const T v = (diag_stride > 0 ? (r % diag_stride == 0) : (r % 2 == 0)) ? T(1) : T(0);
        dst[lqx_layout_offset(s, r, nreal, Vec128<T>::W)] = v;
    }
}
int fill(lqx_ctx* ctx, lqx_field* f) {
    const int V = ctx->geo.V, nreal = 2 * (int)f->kind;
    const int diag = f->kind == LQX_COLORMAT ? 8 : 0;  // reals 0, 8, 16 = the real parts of the diagonal
    if (f->prec == LQX_F32) k_fill_unit<float><<<(V + 127) / 128, 128, 0, ctx->stream>>>(V, nreal, (float*)f->data, diag);
    else k_fill_unit<double><<<(V + 127) / 128, 128, 0, ctx->stream>>>(V, nreal, (double*)f->data, diag);
    return cudaGetLastError() == cudaSuccess ? LQX_OK : LQX_ECUDA;
}

struct Timer {
    lqx_ctx* ctx;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    explicit Timer(lqx_ctx* c) : ctx(c) {
        cudaEventCreate(&e0);
        cudaEventCreate(&e1);
    }
    ~Timer() {
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
    }
    // median device time of fn() over reps launches after one warm-up; < 0 on error
    template <typename F>
    double median_ms(F fn, int reps) {
        if (fn() != LQX_OK) return -1.0;
        std::vector<float> t;
        for (int r = 0; r < reps; ++r) {
            cudaEventRecord(e0, ctx->stream);
            if (fn() != LQX_OK) return -1.0;
            cudaEventRecord(e1, ctx->stream);
            if (cudaEventSynchronize(e1) != cudaSuccess) return -1.0;
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            t.push_back(ms);
        }
        std::sort(t.begin(), t.end());
        return t[t.size() / 2];
    }
};

struct Saved {  // the caller's explicit options are restored whatever happens
    lqx_ctx* c;
    int variant, tile, plaq, hop, jb, js;
    bool timing;
    explicit Saved(lqx_ctx* ctx)
        : c(ctx), variant(ctx->opt_smear_variant), tile(ctx->opt_tile), plaq(ctx->opt_plaq_variant), hop(ctx->opt_hop_block),
          jb(ctx->opt_jacobi_block), js(ctx->opt_jacobi_sites), timing(ctx->timing) {
        ctx->timing = false;
    }
    ~Saved() {
        c->opt_smear_variant = variant, c->opt_tile = tile, c->opt_plaq_variant = plaq, c->opt_hop_block = hop;
        c->opt_jacobi_block = jb, c->opt_jacobi_sites = js, c->timing = timing;
    }
};

}  // namespace

extern "C" int lqx_autotune(lqx_ctx* ctx, int kernel_class, lqx_prec prec, int reps, lqx_tune_row* rows, int max_rows, int* nrows) {
    if (!ctx || (prec != LQX_F32 && prec != LQX_F64) || reps < 1) return LQX_EINVAL;
    if (nrows) *nrows = 0;
    LQX_CUDA(ctx, cudaSetDevice(ctx->device));
    const int pi = prec == LQX_F32 ? 0 : 1;
    Scratch sc;
    Saved saved(ctx);
    Timer timer(ctx);
    std::vector<lqx_tune_row> table;
    auto add = [&](int p0, int p1, double ms) {
        lqx_tune_row r;
        r.kernel_class = kernel_class, r.prec = (int)prec, r.param[0] = p0, r.param[1] = p1, r.ms = ms, r.chosen = 0;
        table.push_back(r);
    };
    lqx_field* u[4];
    for (int mu = 0; mu < 4; ++mu) {
        u[mu] = sc.get(ctx, LQX_COLORMAT, prec);
        if (!u[mu]) return lqx_fail(ctx, LQX_ENOMEM, "autotune: scratch fields");
        if (fill(ctx, u[mu])) return lqx_fail(ctx, LQX_ECUDA, "autotune: fill");
    }
    if (kernel_class == LQX_K_SMEAR) {
        lqx_field* o[4];
        for (int mu = 0; mu < 4; ++mu)
            if (!(o[mu] = sc.get(ctx, LQX_COLORMAT, prec))) return lqx_fail(ctx, LQX_ENOMEM, "autotune: scratch fields");
        // (variant, tile): the literal kernel on row tiles (fp32) and on 4-d tiles / linear blocks.  The other variants
        // are measured slower on every lattice tried and are options, not candidates.
        static const int cand32[][2] = {{10, 1}, {9, 1}, {9, 2}, {3, 1}, {3, 2}, {3, 4}, {3, 5}, {3, 0}};
        static const int cand64[][2] = {{3, 0}, {3, 2}, {3, 3}, {3, 5}, {9, 1}};
        const int(*cand)[2] = pi == 0 ? cand32 : cand64;
        const int ncand = pi == 0 ? (int)(sizeof(cand32) / sizeof(cand32[0])) : (int)(sizeof(cand64) / sizeof(cand64[0]));
        for (int k = 0; k < ncand; ++k) {
            ctx->opt_smear_variant = cand[k][0], ctx->opt_tile = cand[k][1];
            // timed WITH the fused input plaquette, the form the iterated smearing launches (its per-CTA reduction costs the
            // kernels differently: without it the fp64 rolled kernel measured 2.5 % ahead of the row-tile kernel, with it 6 % behind)
            const double ms = timer.median_ms([&] { return lqx_smear_launch(ctx, o, u, 0.5, -1, ctx->h_result); }, reps);
            // a variant that fell back to another kernel on this lattice is not a candidate of its own
            if (ms > 0 && ctx->last_smear_variant == cand[k][0]) add(cand[k][0], cand[k][1], ms);
        }
    } else if (kernel_class == LQX_K_PLAQUETTE) {
        for (int v = 1; v <= 2; ++v) {
            ctx->opt_plaq_variant = v;
            double p;
            const double ms = timer.median_ms([&] { return lqx_plaquette(u, &p, nullptr); }, reps);
            if (ms > 0) add(v, 0, ms);
        }
    } else if (kernel_class == LQX_K_HOP) {
        // param[0] > 0: lqx_hop with that CTA size; param[0] < 0: one iteration of lqx_jacobi_smear with
        // N_threads = -param[0] and N_site = param[1] (the paper's two geometry parameters)
        lqx_field* psi = sc.get(ctx, LQX_FERMION, prec);
        lqx_field* chi = sc.get(ctx, LQX_FERMION, prec);
        lqx_field* t0 = sc.get(ctx, LQX_FERMION, prec);
        lqx_field* t1 = sc.get(ctx, LQX_FERMION, prec);
        if (!psi || !chi || !t0 || !t1) return lqx_fail(ctx, LQX_ENOMEM, "autotune: scratch fields");
        if (fill(ctx, psi) || fill(ctx, chi)) return lqx_fail(ctx, LQX_ECUDA, "autotune: fill");
        for (int b : {32, 64, 128, 256}) {
            ctx->opt_hop_block = b;
            const double ms = timer.median_ms([&] { return lqx_hop(chi, u, psi); }, reps);
            if (ms > 0) add(b, 0, ms);
        }
        lqx_field* tmp[2] = {t0, t1};
        const int iters = 4;
        for (int b : {32, 64, 128, 256})
            for (int ns : {1, 2, 4}) {
                ctx->opt_jacobi_block = b, ctx->opt_jacobi_sites = ns;
                const double ms = timer.median_ms([&] { return lqx_jacobi_smear(chi, u, 0.01, iters, -1, 1.0, tmp); }, reps);
                if (ms > 0) add(-b, ns, ms / iters);
            }
    } else {
        return lqx_fail(ctx, LQX_EINVAL, "autotune: kernel class must be LQX_K_SMEAR, LQX_K_PLAQUETTE or LQX_K_HOP");
    }
    if (table.empty()) return lqx_fail(ctx, LQX_ECUDA, "autotune: no candidate ran");
    // keep the winners
    auto best_of = [&](bool (*pred)(const lqx_tune_row&)) {
        int best = -1;
        for (size_t k = 0; k < table.size(); ++k)
            if (pred(table[k]) && (best < 0 || table[k].ms < table[best].ms)) best = (int)k;
        if (best >= 0) table[best].chosen = 1;
        return best;
    };
    if (kernel_class == LQX_K_SMEAR) {
        const int b = best_of([](const lqx_tune_row&) { return true; });
        ctx->tuned_smear_variant[pi] = table[b].param[0], ctx->tuned_smear_tile[pi] = table[b].param[1];
    } else if (kernel_class == LQX_K_PLAQUETTE) {
        const int b = best_of([](const lqx_tune_row&) { return true; });
        ctx->tuned_plaq_variant[pi] = table[b].param[0];
    } else {
        const int h = best_of([](const lqx_tune_row& r) { return r.param[0] > 0; });
        const int j = best_of([](const lqx_tune_row& r) { return r.param[0] < 0; });
        if (h >= 0) ctx->tuned_hop_block[pi] = table[h].param[0];
        if (j >= 0) ctx->tuned_jacobi_block[pi] = -table[j].param[0], ctx->tuned_jacobi_sites[pi] = table[j].param[1];
    }
    const int n = (int)std::min<size_t>(table.size(), (size_t)std::max(0, max_rows));
    if (rows)
        for (int k = 0; k < n; ++k) rows[k] = table[k];
    if (nrows) *nrows = (int)table.size();
    return LQX_OK;
}

extern "C" int lqx_tuned(const lqx_ctx* ctx, int kernel_class, lqx_prec prec, int out[4]) {
    if (!ctx || !out || (prec != LQX_F32 && prec != LQX_F64)) return LQX_EINVAL;
    const int pi = prec == LQX_F32 ? 0 : 1;
    out[0] = out[1] = out[2] = out[3] = 0;
    if (kernel_class == LQX_K_SMEAR) out[0] = ctx->tuned_smear_variant[pi], out[1] = ctx->tuned_smear_tile[pi];
    else if (kernel_class == LQX_K_PLAQUETTE) out[0] = ctx->tuned_plaq_variant[pi];
    else if (kernel_class == LQX_K_HOP)
        out[0] = ctx->tuned_hop_block[pi], out[1] = ctx->tuned_jacobi_block[pi], out[2] = ctx->tuned_jacobi_sites[pi];
    else return LQX_EINVAL;
    return LQX_OK;
}
