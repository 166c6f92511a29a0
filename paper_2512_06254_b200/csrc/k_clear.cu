// k_clear.cu -- sparse clear of the gridding grid and of the density map.
//
// A snapshot's windows reach a fraction of the G x G cells (a quarter of the 128 x 8-cell tiles at
// config 2, about a tenth at config 4), so zero-filling the whole grid for every snapshot (134 MB of HBM writes at config 2,
// 2.1 GB at config 4) is wasted traffic.  The gridder and the density pass mark the 128 x 8-cell
// tiles they may write in a byte map; once the first FFT pass has read the grid (out of place, into
// the FFT workspace) this kernel zeroes exactly those tiles again and resets the map, so the next
// snapshot finds a zero grid.  The grid is zero-filled in full once, at plan creation.
#include "toi_internal.cuh"

namespace toi {
namespace {

// the work of one warp: clear_tiles_warp (toi_internal.cuh), shared with the transform's column pass
__global__ void __launch_bounds__(256)
k_clear_tiles(float2 *__restrict__ grid, float *__restrict__ dens, int G, uint8_t *__restrict__ map, int tpr,
              long long n_tiles, bool reset)
{
    pdl_wait();
    pdl_trigger();
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    clear_tiles_warp(grid, dens, G, map, tpr, n_tiles, warp * kClearTilesPerWarp, threadIdx.x & 31, reset);
}

}  // namespace

// grid and / or density map (whichever is not null): zero the tiles marked in d_map, reset the map
// (reset_map == false: leave it for a second launch, as the timed path does to time the two apart)
void launch_clear_tiles(float2 *d_grid, float *d_density, int G, uint8_t *d_map, cudaStream_t stream, bool reset_map)
{
    const int tpr = tiles_per_row(G);
    const long long n_tiles = (long long)tpr * tile_rows(G);
    const long long warps = (n_tiles + kClearTilesPerWarp - 1) / kClearTilesPerWarp;
    launch_pdl(k_clear_tiles, dim3((unsigned)((warps + 7) / 8)), dim3(256), 0, stream, d_grid, d_density, G, d_map, tpr, n_tiles, reset_map);
}

}  // namespace toi
