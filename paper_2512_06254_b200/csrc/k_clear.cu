// k_clear.cu -- sparse clear of the gridding grid and of the density map.
//
// A snapshot touches 2-3 % of the G x G cells (3091 of 16384 32x32 tiles at
// config 2), so zero-filling the whole grid for every snapshot (134 MB of HBM writes at config 2,
// 2.1 GB at config 4) is wasted traffic.  The gridder and the density pass mark the 128 x 8-cell
// tiles they may write in a byte map; once the first FFT pass has read the grid (out of place, into
// the FFT workspace) this kernel zeroes exactly those tiles again and resets the map, so the next
// snapshot finds a zero grid.  The grid is zero-filled in full once, at plan creation.
#include "toi_internal.cuh"

namespace toi {
namespace {

// One warp takes kTilesPerWarp consecutive map entries and clears the marked tiles one after the
// other (few tiles per warp: the marked tiles cluster around the uv origin, and a warp that finds
// all of its entries marked must not become the tail of the kernel).  A tile row of the grid is
// kTileW complex64 = 1 KB, written with 8-byte stores.
//
// The density map (uniform weighting) needs no map of its own: the density pass writes the centre
// cells of the samples -- inside the tiles the gridder marks for the same samples' windows -- and
// their mirror cells (-iu, -iv), i.e. array index (G - x, G - y) for (x, y).  For every marked tile
// the same rectangle of the density map and its point mirror are zeroed (4-byte stores: the mirrored
// rectangle starts on any column).
constexpr int kTilesPerWarp = 4;

__global__ void __launch_bounds__(256)
k_clear_tiles(float2 *__restrict__ grid, float *__restrict__ dens, int G, uint8_t *__restrict__ map, int tpr,
              long long n_tiles)
{
    pdl_wait();
    pdl_trigger();
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long t0 = warp * kTilesPerWarp;
    if (t0 >= n_tiles) return;
    const long long mine = t0 + lane;
    const bool dirty = lane < kTilesPerWarp && mine < n_tiles && map[mine] != 0;
    if (dirty) map[mine] = 0;
    unsigned todo = __ballot_sync(0xffffffffu, dirty);
    while (todo) {
        const int b = __ffs(todo) - 1;
        todo &= todo - 1;
        const long long t = t0 + b;
        const int x0 = (int)(t % tpr) * kTileW, y0 = (int)(t / tpr) * kTileH;
        const int rows = min(kTileH, G - y0);
        float2 *row = grid + (size_t)y0 * G + x0;
        for (int r = 0; r < rows; ++r, row += G) {
#pragma unroll
            for (int k = 0; k < kTileW / 32; ++k)
                if (x0 + k * 32 + lane < G) row[k * 32 + lane] = make_float2(0.0f, 0.0f);
        }
        if (dens != nullptr) {
            for (int r = 0; r < rows; ++r) {
                float *own = dens + (size_t)(y0 + r) * G;
                const int ym = G - (y0 + r);                      // mirrored row; G itself is outside
                float *mir = dens + (size_t)(ym < G ? ym : 0) * G;
#pragma unroll
                for (int k = 0; k < kTileW / 32; ++k) {
                    const int x = x0 + k * 32 + lane, xm = G - x;
                    if (x < G) own[x] = 0.0f;
                    if (x < G && ym < G && xm < G) mir[xm] = 0.0f;
                }
            }
        }
    }
}

}  // namespace

// grid (and density map if not null): zero the tiles marked in d_map, reset the map
void launch_clear_tiles(float2 *d_grid, float *d_density, int G, uint8_t *d_map, cudaStream_t stream)
{
    const int tpr = tiles_per_row(G);
    const long long n_tiles = (long long)tpr * tile_rows(G);
    const long long warps = (n_tiles + kTilesPerWarp - 1) / kTilesPerWarp;
    launch_pdl(k_clear_tiles, dim3((unsigned)((warps + 7) / 8)), dim3(256), 0, stream, d_grid, d_density, G, d_map, tpr, n_tiles);
}

}  // namespace toi
