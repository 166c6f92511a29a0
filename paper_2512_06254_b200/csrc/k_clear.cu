// k_clear.cu -- sparse clear of the gridding grid and of the density map.
//
// A snapshot touches 2-3 % of the G x G cells (3091 of 16384 32x32 tiles at
// config 2), so zero-filling the whole grid for every snapshot (134 MB of HBM writes at config 2,
// 2.1 GB at config 4) is wasted traffic.  The gridder and the density pass mark the 32 x 32-cell
// tiles they may write in a byte map; once the first FFT pass has read the grid (out of place, into
// the FFT workspace) this kernel zeroes exactly those tiles again and resets the map, so the next
// snapshot finds a zero grid.  The grid is zero-filled in full once, at plan creation.
#include "toi_internal.cuh"

namespace toi {
namespace {

// One warp takes kTilesPerWarp consecutive map entries and clears the marked tiles one after the
// other (few tiles per warp: the marked tiles cluster around the uv origin, and a warp that finds
// all of its entries marked must not become the tail of the kernel): a tile row is kTile elements
// = 32 x 8 B (complex64) or 16 x 8 B (float32) -- 8-byte stores keep every even G legal (a row
// pitch of G * 4 B is then only 8-byte aligned).
constexpr int kTilesPerWarp = 4;

template <typename T>
__global__ void __launch_bounds__(256)
k_clear_tiles(T *__restrict__ buf, int G, uint8_t *__restrict__ map, int tpr)
{
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long t0 = warp * kTilesPerWarp;
    const long long n_tiles = (long long)tpr * tpr;
    if (t0 >= n_tiles) return;
    const long long mine = t0 + lane;
    const bool dirty = lane < kTilesPerWarp && mine < n_tiles && map[mine] != 0;
    if (dirty) map[mine] = 0;
    unsigned todo = __ballot_sync(0xffffffffu, dirty);
    constexpr int kPerStore = 8 / (int)sizeof(T);                 // elements per 8-byte store: 1 or 2
    constexpr int kLanesPerRow = kTile / kPerStore;               // 32 or 16
    constexpr int kRowsPerPass = 32 / kLanesPerRow;               // 1 or 2
    while (todo) {
        const int b = __ffs(todo) - 1;
        todo &= todo - 1;
        const long long t = t0 + b;
        const int ty = (int)(t / tpr), tx = (int)(t % tpr);
        const int col = tx * kTile + (lane % kLanesPerRow) * kPerStore;
        if (col >= G) continue;                                   // G even: an 8-byte store never straddles the edge
        const int r0 = lane / kLanesPerRow;
        const int rows = min(kTile, G - ty * kTile);
        uint2 *p = reinterpret_cast<uint2 *>(buf + (size_t)(ty * kTile + r0) * G + col);
        const size_t pitch = (size_t)kRowsPerPass * G * sizeof(T) / sizeof(uint2);
#pragma unroll 8
        for (int r = r0; r < rows; r += kRowsPerPass, p += pitch) *p = make_uint2(0u, 0u);
    }
}

}  // namespace

void launch_clear_tiles(float2 *d_grid, int G, uint8_t *d_map, cudaStream_t stream)
{
    const int tpr = tiles_per_row(G);
    const long long warps = ((long long)tpr * tpr + kTilesPerWarp - 1) / kTilesPerWarp;
    k_clear_tiles<float2><<<(unsigned)((warps + 7) / 8), 256, 0, stream>>>(d_grid, G, d_map, tpr);
}

void launch_clear_tiles(float *d_density, int G, uint8_t *d_map, cudaStream_t stream)
{
    const int tpr = tiles_per_row(G);
    const long long warps = ((long long)tpr * tpr + kTilesPerWarp - 1) / kTilesPerWarp;
    k_clear_tiles<float><<<(unsigned)((warps + 7) / 8), 256, 0, stream>>>(d_density, G, d_map, tpr);
}

}  // namespace toi
