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

// scalar path: any even N
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

// vector path, N a multiple of 8: one thread = 4 consecutive pixels of a row (two 16-byte loads of
// F, one 16-byte store); the row factor 1 / (psi(m) omega Wsum) is formed once per thread in fp64,
// the column factors come from the fp64 table, the products are fp32 (two roundings, ~1e-7).
__global__ void __launch_bounds__(256)
k_correct_crop4(int N, int G, const float2 *__restrict__ F, const double *__restrict__ ipsi,
                const SnapState *__restrict__ st, int apply_jacobian, float *__restrict__ image)
{
    const int i = (blockIdx.x * 64 + (threadIdx.x & 63)) * 4;
    const int j = blockIdx.y * 4 + (threadIdx.x >> 6);
    if (i >= N || j >= N) return;
    const double wsum = st->wsum;
    float4 out = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    if (st->status == TOI_OK && wsum > 0.0) {
        const double norm = (apply_jacobian ? st->omega : 1.0) * wsum;
        const int n = i - (N >> 1), m = j - (N >> 1);
        const float4 *src = reinterpret_cast<const float4 *>(F + (size_t)(m < 0 ? m + G : m) * G + (n < 0 ? n + G : n));
        const float4 f01 = __ldg(src), f23 = __ldg(src + 1);
        float row = (float)(ipsi[j] / norm);
        if ((n + m) & 1) row = -row;                       // (-1)^(n+m) of the centred grid
        const double2 c01 = *reinterpret_cast<const double2 *>(ipsi + i), c23 = *reinterpret_cast<const double2 *>(ipsi + i + 2);
        out.x = f01.x * ((float)c01.x * row);
        out.y = -(f01.z * ((float)c01.y * row));
        out.z = f23.x * ((float)c23.x * row);
        out.w = -(f23.z * ((float)c23.y * row));
    }
    *reinterpret_cast<float4 *>(image + (size_t)j * N + i) = out;
}

}  // namespace

void launch_correct_crop(const Geometry &g, const float2 *d_F, const double *d_ipsi, const SnapState *st,
                         int apply_jacobian, float *d_image, cudaStream_t stream)
{
    if (g.N % 8 == 0) {
        dim3 grid((g.N / 4 + 63) / 64, (g.N + 3) / 4);
        k_correct_crop4<<<grid, 256, 0, stream>>>(g.N, g.G, d_F, d_ipsi, st, apply_jacobian, d_image);
    } else {
        dim3 grid((g.N + 31) / 32, (g.N + 7) / 8);
        k_correct_crop<<<grid, 256, 0, stream>>>(g.N, g.G, d_F, d_ipsi, st, apply_jacobian, d_image);
    }
}

}  // namespace toi
