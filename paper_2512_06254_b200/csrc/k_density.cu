// k_density.cu -- step a4 (uniform weighting, reading G14; not in the paper, which
// images with natural weights): density of Stokes-I weight on the gridding cells,
//     D[iv][iu] += w_I   and   D[-iv][-iu] += w_I      (Hermitian-symmetrised)
// Consecutive channels of a baseline share a centre cell for many samples, so each warp takes 32
// consecutive channels, sums w_I over every run of equal cells with a segmented shuffle scan and
// issues ONE reduction per run and mirror instead of one per sample.
#include "toi_internal.cuh"

namespace toi {
namespace {

__global__ void __launch_bounds__(256)
k_density(Geometry g, Inputs in, const SnapState *__restrict__ st, float *__restrict__ D)
{
    if (st->status != TOI_OK) return;
    const int lane = threadIdx.x & 31;
    const int chunks = (g.n_c + 31) >> 5;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (warp >= (long long)g.n_b * chunks) return;
    const int j = (int)(warp / chunks), c = (int)(warp % chunks) * 32 + lane;
    double rho1, rho2;
    rotate_baseline(st->V, in.uvw + 3 * j, rho1, rho2);
    int iu = kOffGrid, iv = kOffGrid;
    float w = 0.0f;
    if (c < g.n_c) {
        float xu, xv;
        sample_cell(rho1, rho2, g.s[c], g.kappa, iu, iv, xu, xv);
        if (cell_on_grid(iu, iv, g.G)) {
            float wa, wb;
            sample_weights(g, in, ((long long)j * g.n_c + c) * g.n_p, wa, wb);
            w = wa + wb;
        } else {
            iu = iv = kOffGrid;
        }
    }
    // segmented inclusive scan over lanes: a run = maximal stretch of lanes with equal (iu, iv)
    const int pu = __shfl_up_sync(0xffffffffu, iu, 1), pv = __shfl_up_sync(0xffffffffu, iv, 1);
    const bool head = lane == 0 || pu != iu || pv != iv;
    const unsigned heads = __ballot_sync(0xffffffffu, head);
    const int start = 31 - __clz(heads & (0xffffffffu >> (31 - lane)));   // my run's first lane
    float sum = w;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const float other = __shfl_up_sync(0xffffffffu, sum, d);
        if (lane - d >= start) sum += other;
    }
    const bool tail = lane == 31 || ((heads >> (lane + 1)) & 1u);
    if (tail && iu != kOffGrid && sum > 0.0f) {
        atomicAdd(D + centre_index(iu, iv, g.G), sum);
        atomicAdd(D + centre_index(-iu, -iv, g.G), sum);
    }
}

}  // namespace

void launch_density(const Geometry &g, const Inputs &in, SnapState *st, float *d_density, cudaStream_t stream)
{
    const long long warps = (long long)g.n_b * ((g.n_c + 31) / 32);
    const int threads = 256;
    const long long blocks = (warps * 32 + threads - 1) / threads;
    k_density<<<(unsigned)blocks, threads, 0, stream>>>(g, in, st, d_density);
}

}  // namespace toi
