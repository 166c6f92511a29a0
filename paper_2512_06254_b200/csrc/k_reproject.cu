// k_reproject.cu -- the re-projection ("interpolate") stage of TOI, PAPER.md:156-200 (section 3.3,
// Eqs. 9-16; Appendix A), and the difference image of two snapshots
// (PAPER.md:83).  The dirty image of the 2-D reconstruction lies on the tilted (t1, t2) plane; it is
// resampled onto the standard (l, m) grid.
//
// Readings (G20-G23): GATHER -- output pixel (i, j) is the direction
// (l, m) = (-beta (i - N/2), +beta (j - N/2)); with q = l^2 + m^2 and z = 1 - n = q / (1 + sqrt(1 - q))
// (Eq. 13) its place on the tilted image is
//     exact (Eqs. 3-4, t = V s):   t1 = V11 l + V12 m - V13 z,   t2 = V21 l + V22 m - V23 z
//     paper (Eqs. 14-15):          t1 = l + xi z,  t2 = m + eta z,  xi = V31/V33, eta = V32/V33
//     p1' = N/2 - t1/beta,  p2' = N/2 + t2/beta                                   (Eq. 16)
// so both are ONE kernel with a 2 x 3 coefficient matrix chosen from V on the device.  The value is
// the bilinear interpolation of the four neighbours; positions outside [0, N-1]^2 (beyond 1e-6 px)
// or outside the SIN domain q <= 1 give NaN.
//
// sm_100a: HBM-bound by design (reads N^2 x 4 B once -- the map is near-affine, so the four taps of
// neighbouring threads fall in the same or adjacent 128-B lines and are served by L1 -- writes
// N^2 x 4 B).  Coordinates are fp64 (a pixel position must be good to ~1e-7 px at N = 8192, which
// fp32 cannot hold); the row/column-separable parts are hoisted (per-thread column terms, per-row
// terms once), leaving one fp64 sqrt, one fp64 divide and a handful of DFMA per pixel.  One thread
// makes 4 consecutive pixels of a row and stores them as one 16-byte vector.
#include <math_constants.h>

#include "toi_internal.cuh"

namespace toi {
namespace {

struct Map {
    double m[6];       // t1 = m0 l + m1 m + m2 z,  t2 = m3 l + m4 m + m5 z
    int ok;
};

__device__ __forceinline__ Map make_map(const double *V, int mode, int status)
{
    Map M;
    M.ok = status == TOI_OK;
    if (mode == TOI_REPROJECT_PAPER) {
        const double xi = V[6] / V[8], eta = V[7] / V[8];          // Eq. 14
        M.m[0] = 1.0; M.m[1] = 0.0; M.m[2] = xi;
        M.m[3] = 0.0; M.m[4] = 1.0; M.m[5] = eta;
    } else {
        M.m[0] = V[0]; M.m[1] = V[1]; M.m[2] = -V[2];
        M.m[3] = V[3]; M.m[4] = V[4]; M.m[5] = -V[5];
    }
    return M;
}

__device__ __forceinline__ float sample_bilinear(const float *__restrict__ src, int N, double p1, double p2, bool valid)
{
    const double hi = (double)(N - 1), eps = 1e-6;
    if (!(valid && p1 >= -eps && p1 <= hi + eps && p2 >= -eps && p2 <= hi + eps)) return CUDART_NAN_F;
    p1 = fmin(fmax(p1, 0.0), hi);
    p2 = fmin(fmax(p2, 0.0), hi);
    const int i0 = min((int)p1, N - 2), j0 = min((int)p2, N - 2);   // p >= 0: truncation is floor
    const float fx = (float)(p1 - (double)i0), fy = (float)(p2 - (double)j0);
    const float *r0 = src + (size_t)j0 * N + i0, *r1 = r0 + N;
    const float a = __ldg(r0), b = __ldg(r0 + 1), c = __ldg(r1), d = __ldg(r1 + 1);
    const float top = fmaf(fx, b - a, a), bot = fmaf(fx, d - c, c);
    return fmaf(fy, bot - top, top);
}

template <int PIX>
__global__ void __launch_bounds__(256)
k_reproject(int N, double beta_rad, const SnapState *__restrict__ st, const double *__restrict__ V_in, int mode,
            const float *__restrict__ src, float *__restrict__ dst)
{
    const int i_base = (blockIdx.x * 64 + (threadIdx.x & 63)) * PIX;
    const int j = blockIdx.y * 4 + (threadIdx.x >> 6);
    if (i_base >= N || j >= N) return;
    const Map M = make_map(V_in ? V_in : st->V, mode, V_in ? TOI_OK : st->status);
    const double inv_beta = 1.0 / beta_rad, half = (double)(N >> 1);
    const double m_ = beta_rad * (double)(j - (N >> 1));
    const double mm = m_ * m_, r1 = M.m[1] * m_, r2 = M.m[4] * m_;
    float out[PIX];
#pragma unroll
    for (int k = 0; k < PIX; ++k) {
        const int i = i_base + k;
        const double l = -beta_rad * (double)(i - (N >> 1));
        const double q = fma(l, l, mm);
        const bool valid = M.ok && q <= 1.0 && i < N;
        const double qs = valid ? q : 0.0;
        const double z = qs / (1.0 + sqrt(1.0 - qs));                 // Eq. 13: 1 - n
        const double t1 = fma(M.m[2], z, fma(M.m[0], l, r1));
        const double t2 = fma(M.m[5], z, fma(M.m[3], l, r2));
        out[k] = sample_bilinear(src, N, fma(-t1, inv_beta, half), fma(t2, inv_beta, half), valid);
    }
    float *o = dst + (size_t)j * N + i_base;
    if (PIX == 4) {
        *reinterpret_cast<float4 *>(o) = make_float4(out[0], out[1], out[2], out[3]);
    } else {
#pragma unroll
        for (int k = 0; k < PIX; ++k)
            if (i_base + k < N) o[k] = out[k];
    }
}

__global__ void __launch_bounds__(256) k_difference4(size_t n4, const float4 *__restrict__ a, const float4 *__restrict__ b,
                                                     float4 *__restrict__ out)
{
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n4; k += (size_t)gridDim.x * blockDim.x) {
        const float4 x = __ldg(a + k), y = __ldg(b + k);
        out[k] = make_float4(x.x - y.x, x.y - y.y, x.z - y.z, x.w - y.w);
    }
}

__global__ void __launch_bounds__(256) k_difference1(size_t n, size_t first, const float *__restrict__ a,
                                                     const float *__restrict__ b, float *__restrict__ out)
{
    const size_t k = first + (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) out[k] = a[k] - b[k];
}

}  // namespace

void launch_reproject(int N, double beta_rad, const SnapState *st, const double *d_V, int mode, const float *d_src,
                      float *d_dst, cudaStream_t stream)
{
    if (N % 4 == 0 && ((uintptr_t)d_dst & 15) == 0) {
        dim3 grid((N / 4 + 63) / 64, (N + 3) / 4);
        k_reproject<4><<<grid, 256, 0, stream>>>(N, beta_rad, st, d_V, mode, d_src, d_dst);
    } else {
        dim3 grid((N + 63) / 64, (N + 3) / 4);
        k_reproject<1><<<grid, 256, 0, stream>>>(N, beta_rad, st, d_V, mode, d_src, d_dst);
    }
}

void launch_difference(size_t n, const float *d_a, const float *d_b, float *d_out, int n_sms, cudaStream_t stream)
{
    const bool aligned = (((uintptr_t)d_a | (uintptr_t)d_b | (uintptr_t)d_out) & 15) == 0;
    const size_t n4 = aligned ? n / 4 : 0;
    if (n4) {
        size_t blocks = (n4 + 255) / 256;
        if (blocks > (size_t)n_sms * 8) blocks = (size_t)n_sms * 8;
        k_difference4<<<(unsigned)blocks, 256, 0, stream>>>(n4, (const float4 *)d_a, (const float4 *)d_b, (float4 *)d_out);
    }
    if (n4 * 4 < n) k_difference1<<<(unsigned)((n - n4 * 4 + 255) / 256), 256, 0, stream>>>(n, n4 * 4, d_a, d_b, d_out);
}

}  // namespace toi
