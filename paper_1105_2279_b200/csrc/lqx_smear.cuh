// Declarations shared by the nearest-neighbour translation units (lqx_lattice.cu: hop, plaquette,
// literal smear and the C entry points; lqx_smear.cu: the shared-corner smear kernel).
#pragma once
#include "lqx_internal.cuh"

template <typename T>
struct Links {
    const T* u[4];
};
template <typename T>
struct LinksOut {
    T* u[4];
};

template <typename T>
static inline Links<T> make_links(const lqx_field* const u[4]) {
    Links<T> l;
    for (int mu = 0; mu < 4; ++mu) l.u[mu] = (const T*)u[mu]->data;
    return l;
}

// an updated link, stored with the streaming (evict-first) policy: it is not read again in this launch, and the
// L2 lines it would take are better spent on the input's halo (row-tile kernel fp32: 2.850 -> 2.836 ms at 48^3x96)
template <typename T>
__device__ __forceinline__ void store_mat_cs(T* p, int s, const Mat3<T>& m) {
    T r[18];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            r[2 * (3 * i + j)] = m.re[i][j];
            r[2 * (3 * i + j) + 1] = m.im[i][j];
        }
    store_site<T, 18, true>(p, s, r);
}

// tile shapes the nearest-neighbour kernels are instantiated for (choice 1..6; 0 = Linear fallback).
// Wide-in-x tiles cost fewer L1 wavefronts for the x-shifted operands (a 16-byte-shifted row of
// TX sites touches one extra 128-byte line per row), compact tiles reuse more neighbours in L1.
typedef Tiled<8, 4, 4, 2> TileA;   // 256 threads
typedef Tiled<8, 4, 2, 2> TileB;   // 128 threads
typedef Tiled<4, 4, 4, 2> TileC;   // 128 threads, for L0 % 8 != 0
typedef Tiled<16, 4, 2, 2> TileD;  // 256 threads
typedef Tiled<16, 2, 2, 2> TileE;  // 128 threads
typedef Tiled<32, 2, 2, 2> TileF;  // 256 threads
static const int kNumTiles = 6;
// first shape that divides the lattice (ctx option "tile" forces one if it fits); 0 = Linear
int lqx_pick_tile(const lqx_ctx* ctx, int first_choice);

#define LQX_WITH_MAP(choice, ...)                 \
    switch (choice) {                             \
        case 1: { typedef TileA MAP; __VA_ARGS__ } break;  \
        case 2: { typedef TileB MAP; __VA_ARGS__ } break;  \
        case 3: { typedef TileC MAP; __VA_ARGS__ } break;  \
        case 4: { typedef TileD MAP; __VA_ARGS__ } break;  \
        case 5: { typedef TileE MAP; __VA_ARGS__ } break;  \
        case 6: { typedef TileF MAP; __VA_ARGS__ } break;  \
        default: { typedef Linear MAP; __VA_ARGS__ } break; \
    }

// z-extent (sites) of a slab of the tile visiting order: thick enough that the two re-read z-faces
// are a small fraction, thin enough that three t-slices of a slab stay in L2
static const int kSlabZ = 16;

// One smear step (all four directions, only_mu < 0) or the bare staple sum of one direction
// (only_mu >= 0, written to uout[0]) on the context's stream (lqx_smear.cu).  If plaq != nullptr the
// plaquette sum of the INPUT field lands there (device or pinned host memory).
int lqx_smear_launch(lqx_ctx* ctx, lqx_field* const uout[4], const lqx_field* const uin[4], double alpha, int only_mu,
                     double* plaq);

// One smear step of the time slices [t0, t1) only (default kernel, no plaquette): LQX_OK, a negative status, or 1
// if the tile shape in use does not split at t0 / t1.  The caller guarantees that the input slices t0-1 .. t1
// (periodic) are complete.
int lqx_smear_launch_range(lqx_ctx* ctx, lqx_field* const uout[4], const lqx_field* const uin[4], double alpha, int t0,
                           int t1);

// ... for any t0 < t1 (falls back to linear blocks where the tile shape in use does not split at t0 / t1)
int lqx_smear_launch_range_any(lqx_ctx* ctx, lqx_field* const uout[4], const lqx_field* const uin[4], double alpha, int t0,
                               int t1);

// shared-memory-staged smear step for fp32 (lqx_smear_staged.cu): LQX_OK, a negative status, or 1 if the
// lattice is not a multiple of its 8x2x2x2 tile
int lqx_smear_staged_launch(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, double* plaq);
void lqx_staged_release(lqx_ctx* ctx);

// smear step with the tile's own links in shared memory (lqx_smear_tile.cu, option "smear_variant" = 7):
// LQX_OK, a negative status, or 1 if no tile shape of this kernel divides the lattice
int lqx_smear_tile_launch(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, double* plaq);
int lqx_smear_tile_launch(lqx_ctx* ctx, const Links<double>& in, const LinksOut<double>& out, double c0, double c1, double* plaq);

// fp32 smear step, plane-ordered 42-product evaluation on whole-x-row tiles in shared memory, persistent
// double-buffered CTAs (lqx_smear_rows.cu, option "smear_variant" = 8): LQX_OK, a negative status, or 1 if
// the lattice does not fit
int lqx_smear_rows_launch(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, double* plaq);
// the literal evaluation on the same row tiles, two CTAs per SM (option "smear_variant" = 9)
int lqx_smear_rowlit_launch(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, double* plaq);
int lqx_smear_rowlit_launch(lqx_ctx* ctx, const Links<double>& in, const LinksOut<double>& out, double c0, double c1, double* plaq);
// variant 10: variant 9's per-link evaluation with the upper staples' common factors kept in tensor memory (fp32)
int lqx_smear_rowz_launch(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, double* plaq);
int lqx_smear_rowz_launch_range(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, int t0, int t1);
bool lqx_smear_rowz_fits(const lqx_ctx* ctx);
// the variant a smear step of this precision runs when nothing narrower is asked for: the explicit option, else the
// auto-tuner's choice, else 10 in fp32 where its eight-row tiles are 257-384 threads (full occupancy of registers, shared
// and tensor memory; elsewhere its TMEM columns cost resident CTAs), else 9.  One rule for the whole-lattice step and for
// t-ranges, so that a decomposed step is bit-identical to the single launch.
int lqx_smear_default_variant(const lqx_ctx* ctx, lqx_prec prec);
int lqx_smear_rowlit_launch_range(lqx_ctx* ctx, const Links<float>& in, const LinksOut<float>& out, float c0, float c1, int t0, int t1);
