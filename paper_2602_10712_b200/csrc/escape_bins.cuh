// escape_bins.cuh -- the direction bins of the escape masks (escape_mask.cu builds them, the trace kernels read
// them): a cube map of the sphere, 6 faces x ESC_GRID x ESC_GRID cells.  CUDA path only.
#pragma once
#include <cuda_runtime.h>

#ifndef ESC_GRID_DEF
#define ESC_GRID_DEF 6
#endif
constexpr int ESC_GRID = ESC_GRID_DEF;                  // <= 8: a face's cells fit one 64-bit word while building
constexpr int ESC_BINS = 6 * ESC_GRID * ESC_GRID;      // 216
constexpr int ESC_WORDS = (ESC_BINS + 31) / 32;         // 7 words per side; 2 sides per triangle
constexpr unsigned long long ESC_CELLS = ESC_GRID == 8 ? ~0ULL : (1ULL << ((ESC_GRID * ESC_GRID) & 63)) - 1ULL;

// bin of direction d (any length > 0): face = 2 * major axis + (negative ? 1 : 0), cell from the other two
// coordinates over |major| in axis order.
__device__ __forceinline__ int esc_bin(float dx, float dy, float dz)
{
    const float ax = fabsf(dx), ay = fabsf(dy), az = fabsf(dz);
    int face; float m, s, t;
    if (ax >= ay && ax >= az) { face = dx < 0.0f ? 1 : 0; m = ax; s = dy; t = dz; }
    else if (ay >= az) { face = dy < 0.0f ? 3 : 2; m = ay; s = dx; t = dz; }
    else { face = dz < 0.0f ? 5 : 4; m = az; s = dx; t = dy; }
    const float im = 1.0f / m;
    int is = (int)((s * im + 1.0f) * (0.5f * ESC_GRID)), it = (int)((t * im + 1.0f) * (0.5f * ESC_GRID));
    is = is < 0 ? 0 : (is > ESC_GRID - 1 ? ESC_GRID - 1 : is);
    it = it < 0 ? 0 : (it > ESC_GRID - 1 ? ESC_GRID - 1 : it);
    return face * (ESC_GRID * ESC_GRID) + it * ESC_GRID + is;
}

// true if a ray leaving global triangle position g on the given side (0: the side of e1 x e2, 1: the other) in
// direction d cannot hit anything (its bin is unmarked)
__device__ __forceinline__ bool esc_escapes(const unsigned *__restrict__ esc, long long g, int side, float dx, float dy, float dz)
{
    const int b = esc_bin(dx, dy, dz);
    return ((__ldg(esc + (size_t)g * (2 * ESC_WORDS) + side * ESC_WORDS + (b >> 5)) >> (b & 31)) & 1u) == 0u;
}
