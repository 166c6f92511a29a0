// k_density.cu -- step a4 (uniform weighting, reading G14; not in the paper, which
// images with natural weights): density of Stokes-I weight on the gridding cells,
//     D[iv][iu] += w_I   and   D[-iv][-iu] += w_I      (Hermitian-symmetrised)
// Consecutive channels of a baseline share a centre cell for many samples, so each warp takes 4 x 32
// consecutive channels (all loads issued up front), sums w_I over every run of equal cells with a
// segmented shuffle scan and issues ONE reduction per run and mirror instead of one per sample.
#include "toi_internal.cuh"

namespace toi {
namespace {

constexpr int kChunks = 4;   // 32-channel chunks per warp: all their loads are in flight together

// FAST: n_p = 4, hands (0, 3), weights 16-B aligned and flags 4-B aligned (or absent): one LDG.128 +
// one LDG.32 per sample; otherwise the generic per-hand loads of sample_weights().
template <bool FAST>
__global__ void __launch_bounds__(256)
k_density(Geometry g, Inputs in, const SnapState *__restrict__ st, float *__restrict__ D)
{
    pdl_wait();
    pdl_trigger();
    if (st->status != TOI_OK) return;
    const int lane = threadIdx.x & 31;
    const int per_row = (g.n_c + 32 * kChunks - 1) / (32 * kChunks);
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (warp >= (long long)g.n_b * per_row) return;
    const int j = (int)(warp / per_row), c0 = (int)(warp % per_row) * (32 * kChunks) + lane;
    const long long q_row = (long long)j * g.n_c;

    // every load of the warp's 128 samples first
    double s[kChunks];
    float4 w4[kChunks];
    unsigned fl[kChunks];
#pragma unroll
    for (int u = 0; u < kChunks; ++u) {
        const int c = c0 + 32 * u;
        s[u] = 0.0; w4[u] = make_float4(1.0f, 0.0f, 0.0f, 1.0f); fl[u] = 0u;
        if (c < g.n_c) {
            s[u] = __ldg(g.s + c);
            if (FAST) {
                if (in.weights) w4[u] = __ldcs(reinterpret_cast<const float4 *>(in.weights) + (q_row + c));
                if (in.flags) fl[u] = __ldcs(reinterpret_cast<const unsigned *>(in.flags) + (q_row + c));
            }
        }
    }
    double rho1, rho2;
    rotate_baseline(st->V, in.uvw + 3 * j, rho1, rho2);
    const int G = g.G;
    float *const Dc = D + centre_index(0, 0, G);

#pragma unroll
    for (int u = 0; u < kChunks; ++u) {
        const int c = c0 + 32 * u;
        int iu = kOffGrid, iv = kOffGrid;
        float w = 0.0f;
        if (c < g.n_c) {
            float xu, xv;
            sample_cell(rho1, rho2, s[u], g.kappa, iu, iv, xu, xv);
            if (cell_on_grid(iu, iv, G)) {
                float wa, wb;
                if (FAST) {
                    wa = (weight_ok(w4[u].x) && !(fl[u] & 0x000000ffu)) ? w4[u].x : 0.0f;
                    wb = (weight_ok(w4[u].w) && !(fl[u] & 0xff000000u)) ? w4[u].w : 0.0f;
                } else {
                    sample_weights(g, in, (q_row + c) * g.n_p, wa, wb);
                }
                w = wa + wb;
            } else {
                iu = iv = kOffGrid;
            }
        }
        // segmented inclusive scan over lanes: a run = maximal stretch of lanes with equal (iu, iv)
        // (an off-grid or padding lane takes a key no cell has, G <= 32768: it never joins a run of cell (0, 0))
        const unsigned key = iu == kOffGrid ? 0x80008000u : ((unsigned)iv << 16) | ((unsigned)iu & 0xffffu);
        const unsigned pk = __shfl_up_sync(0xffffffffu, key, 1);
        const bool head = lane == 0 || pk != key;
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
            const long long o = (long long)iv * G + iu;
            atomicAdd(Dc + o, sum);
            atomicAdd(Dc - o, sum);                       // the mirror cell (-iu, -iv)
        }
    }
}

}  // namespace

void launch_density(const Geometry &g, const Inputs &in, SnapState *st, float *d_density, cudaStream_t stream)
{
    const long long warps = (long long)g.n_b * ((g.n_c + 32 * kChunks - 1) / (32 * kChunks));
    const int threads = 256;
    const long long blocks = (warps * 32 + threads - 1) / threads;
    const uintptr_t aw = (uintptr_t)in.weights, af = (uintptr_t)in.flags;
    if (g.n_p == 4 && g.pol_a == 0 && g.pol_b == 3 && (aw & 15) == 0 && (af & 3) == 0)
        launch_pdl(k_density<true>, dim3((unsigned)blocks), dim3(threads), 0, stream, g, in, (const SnapState *)st, d_density);
    else
        launch_pdl(k_density<false>, dim3((unsigned)blocks), dim3(threads), 0, stream, g, in, (const SnapState *)st, d_density);
}

}  // namespace toi
