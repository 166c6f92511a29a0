// k_grid_atomic.cu -- the comparison gridder (TOI_GRIDDER_ATOMIC): one thread per sample, 49
// complex = 98 float global atomics per visibility.  This is the per-visibility-global-atomics
// scheme the sliding-window gridder (k_grid_sliding.cu) replaces; it stays in the tree as the ncu
// comparison point and as a second, structurally different implementation of step a5.
//   grid[iv+dv][iu+du] += f z phi(iu+du-gu) phi(iv+dv-gv)   (G9, G10)
#include "toi_internal.cuh"

namespace toi {
namespace {

__global__ void __launch_bounds__(256)
k_grid_atomic(Geometry g, Inputs in, SnapState *__restrict__ st, const float *__restrict__ D,
              float2 *__restrict__ grid)
{
    if (st->status != TOI_OK) return;
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double wsum = 0.0;
    unsigned n_grid = 0, n_off = 0, n_flag = 0;
    if (q < (long long)g.n_b * g.n_c) {
        const int j = (int)(q / g.n_c), c = (int)(q % g.n_c);
        double rho1, rho2;
        int iu, iv;
        float xu, xv;
        rotate_baseline(st->V, in.uvw + 3 * j, rho1, rho2);
        sample_cell(rho1, rho2, g.s[c], g.kappa, iu, iv, xu, xv);
        if (!cell_on_grid(iu, iv, g.G)) {
            n_off = 1;
        } else {
            float wa, wb;
            sample_weights(g, in, q * g.n_p, wa, wb);
            const float wI = wa + wb;
            if (!(wI > 0.0f)) {
                n_flag = 1;
            } else {
                n_grid = 1;
                float2 z = sample_stokes(g, in, q * g.n_p, wa, wb);
                float f = 1.0f;
                if (D) f = 1.0f / __ldg(D + centre_index(iu, iv, g.G));
                wsum = (double)f * (double)wI;
                z.x *= f; z.y *= f;
                float pu[kW], pv[kW];
                kernel_taps2(xu, xv, pu, pv);
#pragma unroll
                for (int dv = 0; dv < kW; ++dv) {
                    float2 *row = grid + centre_index(iu - kH, iv + dv - kH, g.G);
#pragma unroll
                    for (int du = 0; du < kW; ++du) {
                        const float wt = pu[du] * pv[dv];
                        float2 *cell = row + du;
                        atomicAdd(&cell->x, z.x * wt);
                        atomicAdd(&cell->y, z.y * wt);
                    }
                }
            }
        }
    }
    // one set of counter atomics per warp
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        wsum += __shfl_xor_sync(0xffffffffu, wsum, d);
        n_grid += __shfl_xor_sync(0xffffffffu, n_grid, d);
        n_off += __shfl_xor_sync(0xffffffffu, n_off, d);
        n_flag += __shfl_xor_sync(0xffffffffu, n_flag, d);
    }
    if ((threadIdx.x & 31) == 0) {
        if (wsum != 0.0) atomicAdd(&st->wsum, wsum);
        if (n_grid) atomicAdd(&st->n_gridded, (unsigned long long)n_grid);
        if (n_off) atomicAdd(&st->n_off_grid, (unsigned long long)n_off);
        if (n_flag) atomicAdd(&st->n_flagged, (unsigned long long)n_flag);
    }
}

}  // namespace

void launch_grid_atomic(const Geometry &g, const Inputs &in, SnapState *st, const float *d_density,
                        float2 *d_grid, cudaStream_t stream)
{
    const long long S = (long long)g.n_b * g.n_c;
    const int threads = 256;
    k_grid_atomic<<<(unsigned)((S + threads - 1) / threads), threads, 0, stream>>>(g, in, st, d_density, d_grid);
}

}  // namespace toi
