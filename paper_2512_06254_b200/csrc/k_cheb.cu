// k_cheb.cu -- helper kernels of the near-coplanar ("3-D") mode, PAPER.md:202-269 (section 3.4,
// Eqs. 17-27): the residual coordinate r3 is kept, its range is cut into slabs, and inside a slab
// the residual phase is expanded in Chebyshev polynomials (Jacobi-Anger, Eqs. 21-22), so that the
// image is a sum of N_slab * K two-dimensional reconstructions ("Chebyshev moments", Eq. 24), each
// made by the ordinary gridder (with the factor T_k(s_q) applied per sample) and cuFFT:
//   I(t1,t2) = Re{ sum_p exp(i 2 pi r3_p t3) sum_k c_k(2 pi Delta_r3 t3) M_pk(t1,t2) } / (omega Wsum)   (Eq. 23)
// Readings: DESIGN.md G24-G26 (equal-width slabs, K rule, valid region = inside the sphere constraint).
//
//   k_r3_range      r3 range of the snapshot (Eq. 26) -- r3 = rho3 * s_c is monotone in s_c, so the
//                   extremes sit at the band edges of the extreme baselines
//   k_cheb_combine  correction + crop of one or two moments (complex: k_correct_crop keeps only Re) fused with
//                   S_p += c_k(alpha) M_pk per pixel, c_0 = J_0, c_k = 2 i^k J_k, and after the slab's last
//                   moment acc += exp(i 2 pi r3_p t3) S_p
//   k_cheb_finish   image = Re(acc) / (omega Wsum); NaN outside the sphere constraint of Eq. 17
#include <math_constants.h>

#include "toi_internal.cuh"

namespace toi {
namespace {

__global__ void __launch_bounds__(256)
k_r3_range(int n_b, const double *__restrict__ uvw, const SnapState *__restrict__ st, double s_min, double s_max,
           double *__restrict__ out /* [2]: r3_min, r3_max */)
{
    __shared__ double s_lo[256], s_hi[256];
    double lo = CUDART_INF, hi = -CUDART_INF;
    for (int j = threadIdx.x; j < n_b; j += blockDim.x) {
        const double rho3 = rotate_row3(st->V, uvw + 3 * j);
        const double a = __dmul_rn(rho3, s_min), b = __dmul_rn(rho3, s_max);   // the gridder's own expression
        lo = fmin(lo, fmin(a, b));
        hi = fmax(hi, fmax(a, b));
    }
    s_lo[threadIdx.x] = lo; s_hi[threadIdx.x] = hi;
    __syncthreads();
    for (int d = 128; d > 0; d >>= 1) {
        if (threadIdx.x < d) {
            s_lo[threadIdx.x] = fmin(s_lo[threadIdx.x], s_lo[threadIdx.x + d]);
            s_hi[threadIdx.x] = fmax(s_hi[threadIdx.x], s_hi[threadIdx.x + d]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[0] = s_lo[0]; out[1] = s_hi[0]; }
}

// t3 of Eq. 17 at pixel (i, j); NaN outside the sphere constraint
__device__ __forceinline__ double t3_pixel(const double *V, int N, double beta_rad, int i, int j)
{
    const double t1 = -beta_rad * (double)(i - (N >> 1)), t2 = beta_rad * (double)(j - (N >> 1));
    const double a = t1 + V[2], b = t2 + V[5];
    const double rad = 1.0 - a * a - b * b;
    if (!(rad >= 0.0)) return CUDART_NAN;
    return -V[8] + (V[8] < 0.0 ? -sqrt(rad) : sqrt(rad));
}

// J_k on a uniform grid of n_tab + 1 points over [-a_max, a_max] (one extra node on each side for
// the 4-point stencil), by the CUDA math library's jn in fp64, stored as K x (n_tab + 3) floats, once per snapshot.
// The combination kernel interpolates it (4-point Lagrange: truncation <= (3/128) h^4 max|d4 J_k| ~ 1e-11
// for h = 2 a_max / 4096, a_max <= ~10; the fp32 table and weights add ~1e-7, against an expansion error
// of 1e-4 .. 1e-2 by Eq. 25) instead of calling jn per pixel and pass, which costs
// several hundred fp64 instructions (a per-pixel Miller recurrence was slower still).
constexpr int kJTab = 4096;

__global__ void __launch_bounds__(256)
k_bessel_table(int K, double a_max, float *__restrict__ tab)
{
    const int m = blockIdx.x * blockDim.x + threadIdx.x;           // 0 .. kJTab + 2
    const int k = blockIdx.y;
    if (m > kJTab + 2 || k >= K) return;
    const double h = 2.0 * a_max / (double)kJTab;
    const double x = -a_max + (double)(m - 1) * h;
    // J_k(-x) = (-1)^k J_k(x); the centre node is x = 0 exactly, where jn(k > 1, 0) returns NaN
    const double v = fabs(x) < 1e-300 ? (k == 0 ? 1.0 : 0.0) : jn(k, fabs(x));
    tab[(size_t)k * (kJTab + 3) + m] = (float)((x < 0.0 && (k & 1)) ? -v : v);
}

// One launch folds NM = 1 or 2 consecutive moments of a slab (orders k0, k0 + 1) into the slab's
// sum S = sum_k i^k c_k(alpha) M_pk (per pixel: t3, the table position and the Lagrange weights are
// computed once for both), and the slab's last launch adds exp(i 2 pi r3_p t3) S to the total -- the
// phase is evaluated once per slab and pixel, not once per moment.
//   first_k: k0 = 0 (S starts at zero);  last_k: k0 + NM = K (S goes into acc instead of back to memory);
//   first_slab: acc starts at zero.
template <int NM>
__global__ void __launch_bounds__(256)
k_cheb_combine(int N, int G, double beta_rad, const SnapState *__restrict__ st, int k0, double r3_p, double d_r3,
               const float *__restrict__ jtab, double a_max, double inv_h, const float2 *__restrict__ F0, const float2 *__restrict__ F1,
               int compact, const double *__restrict__ ipsi, float2 *__restrict__ slab, float2 *__restrict__ acc,
               int first_k, int last_k, int first_slab)
{
    const int i = blockIdx.x * 32 + (threadIdx.x & 31);
    const int j = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (i >= N || j >= N) return;
    const size_t o = (size_t)j * N + i;
    // the moments at this pixel: the transform's unshifted output (compact: already cropped to [j][i]),
    // (-1)^(n+m) of the centred grid, 1/(psi psi).  Everything that does not depend on t3 is requested
    // first, so that its latency runs under the fp64 work below.
    const int n = i - (N >> 1), m = j - (N >> 1);
    const size_t src = compact ? o : (size_t)(m < 0 ? m + G : m) * G + (n < 0 ? n + G : n);
    float2 fm[NM];
    fm[0] = __ldcs(F0 + src);
    if (NM == 2) fm[NM - 1] = __ldcs(F1 + src);
    float2 s = make_float2(0.0f, 0.0f);
    if (!first_k) s = __ldcs(slab + o);
    double c = ipsi[i] * ipsi[j];
    if ((n + m) & 1) c = -c;
    const double t3 = t3_pixel(st->V, N, beta_rad, i, j);
    if (!(t3 == t3)) return;                                             // outside Eq. 17's sphere: k_cheb_finish writes NaN
    const double two_pi = 6.283185307179586476925286766559;
    // Eq. 20: alpha = 2 pi d t3; position in the Bessel table in fp64, the 4-point Lagrange weights on nodes
    // -1, 0, 1, 2 and the interpolation in fp32 (|J_k| <= 1: 1e-7 absolute)
    float w0 = 0.0f, w1 = 0.0f, w2 = 0.0f, w3 = 0.0f;
    int node = 0;
    if (a_max > 0.0) {
        double u = (two_pi * d_r3 * t3 + a_max) * inv_h;                 // 0 .. kJTab
        u = fmin(fmax(u, 0.0), (double)kJTab);
        node = (int)u;
        if (node > kJTab - 1) node = kJTab - 1;
        const float f = (float)(u - (double)node);                       // [0, 1]
        w0 = -f * (f - 1.0f) * (f - 2.0f) * (1.0f / 6.0f);
        w1 = (f + 1.0f) * (f - 1.0f) * (f - 2.0f) * 0.5f;
        w2 = -(f + 1.0f) * f * (f - 2.0f) * 0.5f;
        w3 = (f + 1.0f) * f * (f - 1.0f) * (1.0f / 6.0f);
    }
    const float cf = (float)c;
#pragma unroll
    for (int q = 0; q < NM; ++q) {
        const int k = k0 + q;
        float ck;                                                        // Eq. 22: c_0 = J_0, c_k = 2 J_k (times i^k below)
        if (a_max > 0.0) {
            const float *row = jtab + (size_t)k * (kJTab + 3) + node;    // nodes node-1 .. node+2 (rows are offset by one)
            ck = w0 * __ldg(row) + w1 * __ldg(row + 1) + w2 * __ldg(row + 2) + w3 * __ldg(row + 3);
        } else {
            ck = k == 0 ? 1.0f : 0.0f;                                   // alpha = 0 everywhere
        }
        if (k > 0) ck *= 2.0f;
        const float a = ck * cf;
        const float2 f = fm[q];
        switch (k & 3) {                                                 // s += i^k a f
        case 0: s.x += a * f.x; s.y += a * f.y; break;
        case 1: s.x -= a * f.y; s.y += a * f.x; break;
        case 2: s.x -= a * f.x; s.y -= a * f.y; break;
        default: s.x += a * f.y; s.y -= a * f.x; break;
        }
    }
    if (!last_k) {
        __stcs(slab + o, s);
        return;
    }
    double sp, cp;
    sincospi(2.0 * r3_p * t3, &sp, &cp);                                 // exp(i 2 pi r3_p t3)
    float2 t = first_slab ? make_float2(0.0f, 0.0f) : acc[o];
    t.x += (float)(cp * (double)s.x - sp * (double)s.y);
    t.y += (float)(cp * (double)s.y + sp * (double)s.x);
    acc[o] = t;
}

__global__ void __launch_bounds__(256)
k_cheb_finish(int N, double beta_rad, const SnapState *__restrict__ st, int apply_jacobian,
              const float2 *__restrict__ acc, float *__restrict__ image)
{
    const int i = blockIdx.x * 32 + (threadIdx.x & 31);
    const int j = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (i >= N || j >= N) return;
    const size_t o = (size_t)j * N + i;
    float out = 0.0f;
    const double wsum = st->wsum;
    if (st->status == TOI_OK && wsum > 0.0) {
        const double t3 = t3_pixel(st->V, N, beta_rad, i, j);
        out = (t3 == t3) ? (float)((double)acc[o].x / ((apply_jacobian ? st->omega : 1.0) * wsum)) : CUDART_NAN_F;
    }
    image[o] = out;
}

}  // namespace

void launch_r3_range(int n_b, const double *d_uvw, const SnapState *st, double s_min, double s_max, double *d_out,
                     cudaStream_t stream)
{
    k_r3_range<<<1, 256, 0, stream>>>(n_b, d_uvw, st, s_min, s_max, d_out);
}

size_t bessel_table_floats(int K) { return (size_t)K * (kJTab + 3); }

void launch_bessel_table(int K, double a_max, float *d_tab, cudaStream_t stream)
{
    if (!(a_max > 0.0)) return;
    dim3 grid((kJTab + 3 + 255) / 256, K);
    k_bessel_table<<<grid, 256, 0, stream>>>(K, a_max, d_tab);
}

void launch_cheb_combine(const Geometry &g, double beta_rad, const SnapState *st, int k0, int n_moments, double r3_p,
                         double d_r3, const float *d_tab, double a_max, const float2 *d_F0, const float2 *d_F1, int compact,
                         const double *d_ipsi, float2 *d_slab, float2 *d_acc, int first_k, int last_k, int first_slab,
                         cudaStream_t stream)
{
    dim3 grid((g.N + 31) / 32, (g.N + 7) / 8);
    const double inv_h = a_max > 0.0 ? (double)kJTab / (2.0 * a_max) : 0.0;
    if (n_moments == 2)
        k_cheb_combine<2><<<grid, 256, 0, stream>>>(g.N, g.G, beta_rad, st, k0, r3_p, d_r3, d_tab, a_max, inv_h, d_F0, d_F1, compact,
                                                    d_ipsi, d_slab, d_acc, first_k, last_k, first_slab);
    else
        k_cheb_combine<1><<<grid, 256, 0, stream>>>(g.N, g.G, beta_rad, st, k0, r3_p, d_r3, d_tab, a_max, inv_h, d_F0, d_F0, compact,
                                                    d_ipsi, d_slab, d_acc, first_k, last_k, first_slab);
}

void launch_cheb_finish(int N, double beta_rad, const SnapState *st, int apply_jacobian, const float2 *d_acc,
                        float *d_image, cudaStream_t stream)
{
    dim3 grid((N + 31) / 32, (N + 7) / 8);
    k_cheb_finish<<<grid, 256, 0, stream>>>(N, beta_rad, st, apply_jacobian, d_acc, d_image);
}

}  // namespace toi
