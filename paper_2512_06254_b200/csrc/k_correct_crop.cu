// k_correct_crop.cu -- step a7, fused: grid correction, crop to the central N x N, and the
// normalisation of Eq. 7:
//     image[j][i] = Re F[m][n] / (psi(n) psi(m) omega Wsum),  n = i - N/2, m = j - N/2
// F is cuFFT's unshifted output: pixel offset n lives at array index (n + G) mod G, so the crop is
// four corner blocks of F; the grid went in CENTRED (cell k at index k + G/2), which multiplies F
// by (-1)^(n+m) (shift theorem) -- undone here by the sign.  No fftshift pass exists.  1/psi is tabulated in fp64 at plan time
// (G11); omega and Wsum are read from device memory (no host round trip).
#include "toi_internal.cuh"

namespace toi {
namespace {

__global__ void __launch_bounds__(256)
k_correct_crop(int N, int G, const float2 *__restrict__ F, const double *__restrict__ ipsi,
               const SnapState *__restrict__ st, int apply_jacobian, float *__restrict__ image)
{
    const int i = blockIdx.x * 32 + (threadIdx.x & 31);
    const int j = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (i >= N || j >= N) return;
    const double wsum = st->wsum;
    float out = 0.0f;
    if (st->status == TOI_OK && wsum > 0.0) {
        const double norm = (apply_jacobian ? st->omega : 1.0) * wsum;
        const int n = i - (N >> 1), m = j - (N >> 1);
        const float2 f = __ldg(F + (size_t)(m < 0 ? m + G : m) * G + (n < 0 ? n + G : n));
        const double v = (double)f.x * (ipsi[i] * ipsi[j] / norm);
        out = (float)(((n + m) & 1) ? -v : v);
    }
    image[(size_t)j * N + i] = out;
}

}  // namespace

void launch_correct_crop(const Geometry &g, const float2 *d_F, const double *d_ipsi, const SnapState *st,
                         int apply_jacobian, float *d_image, cudaStream_t stream)
{
    dim3 grid((g.N + 31) / 32, (g.N + 7) / 8);
    k_correct_crop<<<grid, 256, 0, stream>>>(g.N, g.G, d_F, d_ipsi, st, apply_jacobian, d_image);
}

}  // namespace toi
