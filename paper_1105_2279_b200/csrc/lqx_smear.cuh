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

// tile shapes the nearest-neighbour kernels are instantiated for (choice 1..3; 0 = Linear fallback)
typedef Tiled<8, 4, 4, 2> TileA;  // 256 threads
typedef Tiled<8, 4, 2, 2> TileB;  // 128 threads
typedef Tiled<4, 4, 4, 2> TileC;  // 128 threads, for L0 % 8 != 0
// first shape that divides the lattice (ctx option "tile" forces one if it fits); 0 = Linear
int lqx_pick_tile(const lqx_ctx* ctx, int first_choice);

#define LQX_WITH_MAP(choice, ...)                 \
    switch (choice) {                             \
        case 1: { typedef TileA MAP; __VA_ARGS__ } break;  \
        case 2: { typedef TileB MAP; __VA_ARGS__ } break;  \
        case 3: { typedef TileC MAP; __VA_ARGS__ } break;  \
        default: { typedef Linear MAP; __VA_ARGS__ } break; \
    }

// shared-corner smear step (lqx_smear.cu).  Returns LQX_OK, or 1 if this lattice / precision is
// not covered and the caller should use the literal kernel.
int lqx_smear_shared_launch(lqx_ctx* ctx, lqx_field* const uout[4], const lqx_field* const uin[4], double alpha,
                            double* plaq_out);
