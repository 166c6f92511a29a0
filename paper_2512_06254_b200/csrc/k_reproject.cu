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
// terms once); the square root and the quotient of Eq. 13 are 20-bit MUFU.RSQ64H / RCP64H seeds refined
// by one Newton step in fp64 (no library slow paths, no fp64<->fp32 conversions on the quarter-rate
// XU pipe, which bounded the first version): ~26 fp64 instructions and 4 XU instructions per pixel.  One thread makes 4
// consecutive pixels of a row and stores them as one 16-byte vector.
#include <math_constants.h>

#include "toi_internal.cuh"

namespace toi {
namespace {

struct Map {
    double m[6];       // t1 = m0 l + m1 m + m2 z,  t2 = m3 l + m4 m + m5 z
    int ok;
};

// 1/d for d in [1e-6, 4]: MUFU.RCP64H seed (rcp.approx.ftz.f64: ~20 good bits from ONE instruction of
// the quarter-rate XU pipe, where an fp32 seed costs three -- two conversions and the MUFU) + Newton
// steps in fp64 (each squares the error); no special cases can occur in that range, so none of the
// library division's slow paths are carried along.
template <int STEPS>
__device__ __forceinline__ double rcp_newton(double d)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
#pragma unroll
    for (int k = 0; k < STEPS; ++k) r = fma(r, fma(-d, r, 1.0), r);
    return r;
}

__device__ __forceinline__ Map make_map(const double *V, int mode, int status)
{
    Map M;
    M.ok = status == TOI_OK;
    if (mode == TOI_REPROJECT_PAPER) {
        const double r33 = M.ok ? rcp_newton<4>(fabs(V[8])) : 0.0;     // |V33| >= 1e-6 when ok
        const double s33 = V[8] < 0.0 ? -r33 : r33;
        M.m[0] = 1.0; M.m[1] = 0.0; M.m[2] = V[6] * s33;               // Eq. 14: xi
        M.m[3] = 0.0; M.m[4] = 1.0; M.m[5] = V[7] * s33;               //         eta
    } else {
        M.m[0] = V[0]; M.m[1] = V[1]; M.m[2] = -V[2];
        M.m[3] = V[3]; M.m[4] = V[4]; M.m[5] = -V[5];
    }
    return M;
}

// Eq. 13, z = 1 - n = q / (1 + sqrt(1 - q)) for 0 <= q <= 1, relative error ~2e-12 (one Newton
// step on a 20-bit MUFU.RSQ64H seed gives n to 1.5 e0^2, one on a MUFU.RCP64H seed the quotient):
// z / beta is at most ~1e4 pixels, so the position is good to ~1e-8 px.
__device__ __forceinline__ double sin_z(double q)
{
    // + 1e-300: a stays a positive normal number at the horizon (q = 1: n -> 0, z -> 1) and is
    // unchanged everywhere else; q > 1 (outside the SIN domain) gives NaN, which the caller never uses
    const double a = (1.0 - q) + 1e-300;
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(a));
    const double t = a * y0;                               // ~ sqrt(a)
    const double n = fma(0.5 * t, fma(-t, y0, 1.0), t);    // Newton: t (1 + (1 - a y0^2)/2)
    return q * rcp_newton<1>(1.0 + n);
}

// One axis of the bilinear tap: p -> first neighbour i0 in [0, N-2] and weight f in [0, 1] of the
// second; false when p is more than 1e-6 px outside [0, N-1] (G22) or NaN.  floor(p) by the
// magic-number add (round-down add of 2^52 + 2^51 leaves floor(p) in the low word) on the fp64
// pipe instead of two XU conversions; its result is only used when the range test passed.
__device__ __forceinline__ bool tap(double p, int N, int &i0, float &f)
{
    const bool in = p >= -1e-6 && p <= (double)(N - 1) + 1e-6;       // false for NaN
    const double m = __dadd_rd(p, kFloorMagic);
    const int k = __double2loint(m);                                 // -1 .. N-1 when in
    const float w = (float)(p - (m - kFloorMagic));                  // [0, 1)
    i0 = min(max(k, 0), N - 2);
    f = k < 0 ? 0.0f : (k > N - 2 ? 1.0f : w);
    return in;
}

// Narrow fields (launch_reproject checks q <= 1/4 everywhere and |q_k - q_0| <= 1e-5 inside a thread's
// four pixels): Eq. 13 is evaluated exactly (sin_z's route) once per thread, at its first pixel, and
// carried to the other three by the expansion of the square root about it,
//   z(q0 + d) = z0 + n0 e (1/2 + e (1/8 + e / 16)),  e = d / (1 - q0),  n0 = sqrt(1 - q0),
// whose first neglected term is 5 e^4 n0 / 128 < 1e-20: 6 fp64 instructions per pixel instead of 14
// and two MUFU, with the linear parts of Eq. 4 advanced by their per-pixel steps.
template <bool FAST_UNUSED = true>
__global__ void __launch_bounds__(256)
k_reproject_narrow(int N, double beta_rad, const SnapState *__restrict__ st, const double *__restrict__ V_in, int mode,
                   const float *__restrict__ src, float *__restrict__ dst)
{
    const int i_base = (blockIdx.x * 64 + (threadIdx.x & 63)) * 4;
    const int j = blockIdx.y * 4 + (threadIdx.x >> 6);
    if (i_base >= N || j >= N) return;
    const Map M = make_map(V_in ? V_in : st->V, mode, V_in ? TOI_OK : st->status);
    const double inv_beta = 1.0 / beta_rad, half = (double)(N >> 1);
    const double m_ = beta_rad * (double)(j - (N >> 1));
    const double l0 = -beta_rad * (double)(i_base - (N >> 1));
    const double q0 = fma(l0, l0, m_ * m_);
    // n0 = sqrt(1 - q0) and y = 1 / n0 to ~1e-12 (one Newton step on the 20-bit seed), z0 = q0 / (1 + n0)
    const double a0 = 1.0 - q0;
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(a0));
    const double y = fma(0.5 * y0, fma(-a0 * y0, y0, 1.0), y0);
    const double n0 = a0 * y, yy = y * y;
    const double z0 = q0 * rcp_newton<1>(1.0 + n0);
    // linear parts at pixel 0 and their steps per pixel (l_k = l0 - beta k)
    const double A1 = fma(M.m[0], l0, M.m[1] * m_), A2 = fma(M.m[3], l0, M.m[4] * m_);
    const double s1 = -beta_rad * M.m[0], s2 = -beta_rad * M.m[3];
    const double bb = beta_rad * beta_rad, two_bl0 = 2.0 * beta_rad * l0;
    float out[4], fx[4], fy[4];
    int i0[4], j0[4];
    bool ok[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        double z = z0;
        if (k > 0) {
            const double d = (double)k * fma(bb, (double)k, -two_bl0);          // q_k - q_0
            const double e = d * yy;
            z = fma(n0 * e, fma(e, fma(e, 0.0625, 0.125), 0.5), z0);
        }
        const double t1 = fma(M.m[2], z, fma((double)k, s1, A1));
        const double t2 = fma(M.m[5], z, fma((double)k, s2, A2));
        ok[k] = M.ok;
        ok[k] = tap(fma(-t1, inv_beta, half), N, i0[k], fx[k]) && ok[k];
        ok[k] = tap(fma(t2, inv_beta, half), N, j0[k], fy[k]) && ok[k];
    }
    // the taps are clamped into the image whatever the position, so all 16 loads go out together
    // (a branch per pixel serialised them behind one another's latency); invalid pixels become NaN after
    float a[4], b[4], c[4], dd[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float *p0 = src + (size_t)j0[k] * N + i0[k], *p1 = p0 + N;
        a[k] = __ldg(p0); b[k] = __ldg(p0 + 1); c[k] = __ldg(p1); dd[k] = __ldg(p1 + 1);
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float top = fmaf(fx[k], b[k] - a[k], a[k]), bot = fmaf(fx[k], dd[k] - c[k], c[k]);
        out[k] = ok[k] ? fmaf(fy[k], bot - top, top) : CUDART_NAN_F;
    }
    *reinterpret_cast<float4 *>(dst + (size_t)j * N + i_base) = make_float4(out[0], out[1], out[2], out[3]);
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
    const double l0 = -beta_rad * (double)(i_base - (N >> 1));
    float out[PIX], fx[PIX], fy[PIX];
    int i0[PIX], j0[PIX];
    bool ok[PIX];
#pragma unroll
    for (int k = 0; k < PIX; ++k) {
        const double l = fma(-beta_rad, (double)k, l0);
        const double q = fma(l, l, mm);
        const double z = sin_z(fmin(q, 1.0));
        const double t1 = fma(M.m[2], z, fma(M.m[0], l, r1));
        const double t2 = fma(M.m[5], z, fma(M.m[3], l, r2));
        ok[k] = M.ok && q <= 1.0 && i_base + k < N;
        ok[k] = tap(fma(-t1, inv_beta, half), N, i0[k], fx[k]) && ok[k];
        ok[k] = tap(fma(t2, inv_beta, half), N, j0[k], fy[k]) && ok[k];
    }
    // the taps are clamped into the image whatever the position: all loads go out together
#pragma unroll
    for (int k = 0; k < PIX; ++k) {
        const float *p0 = src + (size_t)j0[k] * N + i0[k], *p1 = p0 + N;
        const float a = __ldg(p0), b = __ldg(p0 + 1), c = __ldg(p1), d = __ldg(p1 + 1);
        const float top = fmaf(fx[k], b - a, a), bot = fmaf(fx[k], d - c, c);
        out[k] = ok[k] ? fmaf(fy[k], bot - top, top) : CUDART_NAN_F;
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
        // narrow field: q = l^2 + m^2 <= 1/4 over the image and |q_k - q_0| <= 1e-5 within four pixels
        const double l_max = beta_rad * (0.5 * N + 1.0);
        if (2.0 * l_max * l_max <= 0.25 && 3.0 * beta_rad * (2.0 * l_max + 3.0 * beta_rad) <= 1e-5)
            k_reproject_narrow<><<<grid, 256, 0, stream>>>(N, beta_rad, st, d_V, mode, d_src, d_dst);
        else
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
