// fft_smem.cuh -- power-of-two complex FFT of one sequence held in shared memory, the core of
// the pruned inverse transform of step a6 (k_fft.cu):
//   X[k] = sum_n x[n] exp(+2 pi i n k / G)        (unnormalised, sign +i: PAPER.md:301, DESIGN.md step 8)
// Stockham autosort, decimation in time: stage s with radix R takes the G / R butterflies
//   j = 0 .. G/R - 1,  k = j mod Ns  (Ns = product of the radices of the earlier stages)
//   v[r] = x[j + r G/R] * W^(r k G / (Ns R)),  V = DFT_R(v),  y[(j - k) R + k + r Ns] = V[r]
// with natural order in and out.  G / 16 threads work on one sequence; every thread moves 16
// elements per stage through its registers (16 / R butterflies), all loads of a stage happen before
// its first store (a barrier in between), so the stage runs in place.  Stages: radix 16 as long as
// possible, then one of radix 8, 4 or 2.  The sequence is padded by one element per 16 (stage 1
// stores with a stride of 16 elements: 17 keeps a half-warp of 8-byte stores on 16 different bank pairs).
// Twiddles: W^m = exp(+2 pi i m / G) from a table of G float2 computed in fp64 on the host; per
// butterfly the powers w, w^2, w^4, w^8 of its base twiddle are looked up (from per-stage tables
// in shared memory, 8.5 KB per CTA), the others are products of at most three of them.
#pragma once
#include <cuda_runtime.h>

namespace toi {
namespace fft {

__device__ __forceinline__ int pad(int i) { return i + (i >> 4); }
__host__ __device__ constexpr int padded(int n) { return n + (n >> 4); }

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 muli(float2 a) { return make_float2(-a.y, a.x); }      // * (+i)

__device__ __forceinline__ void dft2(float2 &a, float2 &b)
{
    const float2 t = csub(a, b);
    a = cadd(a, b);
    b = t;
}

// X[k] = sum_n a[n] (+i)^(n k)
__device__ __forceinline__ void dft4(float2 &a0, float2 &a1, float2 &a2, float2 &a3)
{
    const float2 t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = muli(csub(a1, a3));
    a0 = cadd(t0, t2);
    a1 = cadd(t1, t3);
    a2 = csub(t0, t2);
    a3 = csub(t1, t3);
}

// 8 = 2 x 4: n = 2 a + b, k = c + 4 d:  X[c + 4 d] = sum_b (-1)^(b d) W8^(b c) sum_a x[2 a + b] (+i)^(a c)
__device__ __forceinline__ void dft8(float2 *v)
{
    constexpr float h = 0.70710678118654752440f;
    dft4(v[0], v[2], v[4], v[6]);                       // b = 0: Y0[c] in v[0], v[2], v[4], v[6]
    dft4(v[1], v[3], v[5], v[7]);                       // b = 1: Y1[c] in v[1], v[3], v[5], v[7]
    // Y1[c] *= W8^c, W8 = exp(+2 pi i / 8)
    v[3] = make_float2(h * (v[3].x - v[3].y), h * (v[3].x + v[3].y));
    v[5] = muli(v[5]);
    v[7] = make_float2(-h * (v[7].x + v[7].y), h * (v[7].x - v[7].y));
    // X[c] = Y0[c] + Y1[c], X[c + 4] = Y0[c] - Y1[c]
    float2 x[8];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        x[c] = cadd(v[2 * c], v[2 * c + 1]);
        x[c + 4] = csub(v[2 * c], v[2 * c + 1]);
    }
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = x[k];
}

// 16 = 4 x 4: n = 4 a + b, k = c + 4 d:
//   X[c + 4 d] = sum_b (+i)^(b d) [ W16^(b c) sum_a x[4 a + b] (+i)^(a c) ]
__device__ __forceinline__ void dft16(float2 *v)
{
    constexpr float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f, h = 0.70710678118654752440f;
#pragma unroll
    for (int b = 0; b < 4; ++b) dft4(v[b], v[4 + b], v[8 + b], v[12 + b]);      // Y_b[c] in v[4 c + b]
    // Z_b[c] = Y_b[c] W16^(b c), W16^m = (cos, sin)(2 pi m / 16)
    v[5] = cmul(v[5], make_float2(c1, s1));              // b = 1, c = 1: W^1
    v[9] = cmul(v[9], make_float2(h, h));                // b = 1, c = 2: W^2
    v[13] = cmul(v[13], make_float2(s1, c1));            // b = 1, c = 3: W^3
    v[6] = cmul(v[6], make_float2(h, h));                // b = 2, c = 1: W^2
    v[10] = muli(v[10]);                                 // b = 2, c = 2: W^4 = i
    v[14] = cmul(v[14], make_float2(-h, h));             // b = 2, c = 3: W^6
    v[7] = cmul(v[7], make_float2(s1, c1));              // b = 3, c = 1: W^3
    v[11] = cmul(v[11], make_float2(-h, h));             // b = 3, c = 2: W^6
    v[15] = cmul(v[15], make_float2(-c1, -s1));          // b = 3, c = 3: W^9
    float2 x[16];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        float2 z0 = v[4 * c], z1 = v[4 * c + 1], z2 = v[4 * c + 2], z3 = v[4 * c + 3];
        dft4(z0, z1, z2, z3);                            // over b, indexed by d
        x[c] = z0; x[c + 4] = z1; x[c + 8] = z2; x[c + 12] = z3;
    }
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = x[k];
}

template <int R>
__device__ __forceinline__ void dft(float2 *v)
{
    if (R == 16) dft16(v);
    else if (R == 8) dft8(v);
    else if (R == 4) dft4(v[0], v[1], v[2], v[3]);
    else dft2(v[0], v[1]);
}

// v[r] *= w^r, r = 1 .. R - 1, from the powers p[0..3] = {w, w^2, w^4, w^8} of the butterfly's base twiddle
template <int R>
__device__ __forceinline__ void twiddle(float2 *v, const float2 *p)
{
    const float2 w1 = p[0];
    v[1] = cmul(v[1], w1);
    if (R >= 4) {
        const float2 w2 = p[1];
        const float2 w3 = cmul(w1, w2);
        v[2] = cmul(v[2], w2);
        v[3] = cmul(v[3], w3);
        if (R >= 8) {
            const float2 w4 = p[2];
            const float2 w5 = cmul(w1, w4), w6 = cmul(w2, w4), w7 = cmul(w3, w4);
            v[4] = cmul(v[4], w4); v[5] = cmul(v[5], w5); v[6] = cmul(v[6], w6); v[7] = cmul(v[7], w7);
            if (R >= 16) {
                const float2 w8 = p[3];
                v[8] = cmul(v[8], w8); v[9] = cmul(v[9], cmul(w1, w8)); v[10] = cmul(v[10], cmul(w2, w8));
                v[11] = cmul(v[11], cmul(w3, w8)); v[12] = cmul(v[12], cmul(w4, w8)); v[13] = cmul(v[13], cmul(w5, w8));
                v[14] = cmul(v[14], cmul(w6, w8)); v[15] = cmul(v[15], cmul(w7, w8));
            }
        }
    }
}

// Twiddle tables of the stages with NS = 16 and NS = 256, in shared memory: row k holds the powers
// {w, w^2, w^4, w^8} of w = W^(k G / (NS R)) (R = the radix of that stage).  Filled once per CTA from
// the global table W^m = exp(+2 pi i m / G); 16 x 4 + 256 x 4 float2 = 8.5 KB.
constexpr int kTabFloat2 = (16 + 256) * 4;
template <int LOG2G>
__device__ __forceinline__ void fill_tables(float2 *tab, const float2 *__restrict__ tw, int tid, int n_threads)
{
    constexpr int G = 1 << LOG2G;
    constexpr int R3 = LOG2G >= 12 ? 16 : (LOG2G == 11 ? 8 : 4);      // radix of the NS = 256 stage
    for (int e = tid; e < kTabFloat2; e += n_threads) {
        const int k = e >> 2, p = e & 3;
        const int m1 = k < 16 ? k * (G / (16 * 16)) : (k - 16) * (G / (256 * R3));
        tab[e] = __ldg(tw + (((m1 << p)) & (G - 1)));
    }
}

// One stage on the sequence at `s` (padded); t = my index among the G / 16 threads of the sequence.
// Contains two CTA-wide barriers: every thread of the CTA must call it the same number of times.
// `tab`: the shared-memory twiddle rows of this stage (NS = 16, 256) or nullptr (NS = 1: no twiddles;
// NS = 4096: looked up in the global table `tw`, consecutive threads consecutive entries).
// `out`: where the results go -- SmemOut (back into the sequence, followed by a barrier) or a functor
// out(index, value) of the caller's (the last stage of a pass can hand its results straight to global
// memory: consecutive threads hold consecutive indices).
struct SmemOut {
    float2 *s;
    static constexpr bool kShared = true;
    __device__ __forceinline__ void operator()(int i, float2 v) const { s[pad(i)] = v; }
};

template <int R, int G, int NS, class Out>
__device__ __forceinline__ void stage(float2 *s, int t, const float2 *tab, const float2 *__restrict__ tw, const Out &out)
{
    constexpr int T = G / 16, B = 16 / R;
    float2 v[16];
#pragma unroll
    for (int q = 0; q < B; ++q) {
        const int j = t + q * T;
#pragma unroll
        for (int r = 0; r < R; ++r) v[q * R + r] = s[pad(j + r * (G / R))];
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < B; ++q) {
        const int j = t + q * T;
        const int k = j & (NS - 1);
        if (NS == 16 || NS == 256) {
            float2 p[4];
            const float4 lo = *reinterpret_cast<const float4 *>(tab + 4 * k), hi = *reinterpret_cast<const float4 *>(tab + 4 * k + 2);
            p[0] = make_float2(lo.x, lo.y); p[1] = make_float2(lo.z, lo.w);
            p[2] = make_float2(hi.x, hi.y); p[3] = make_float2(hi.z, hi.w);
            twiddle<R>(v + q * R, p);
        } else if (NS > 1) {
            float2 p[4];
            const int m1 = k * (G / (NS * R));
            p[0] = __ldg(tw + m1);
            p[1] = R >= 4 ? __ldg(tw + ((2 * m1) & (G - 1))) : p[0];
            p[2] = p[3] = p[0];
            twiddle<R>(v + q * R, p);
        }
        dft<R>(v + q * R);
        const int j0 = (j - k) * R + k;
#pragma unroll
        for (int r = 0; r < R; ++r) out(j0 + r * NS, v[q * R + r]);
    }
    if (Out::kShared) __syncthreads();
}

// The whole transform: G = 2^LOG2G, 10 <= LOG2G <= 14.  `tab`: fill_tables' output.  The last stage's
// results go to `out` (SmemOut{s}: in place).
template <int LOG2G, class Out>
__device__ __forceinline__ void transform(float2 *s, int t, const float2 *tab, const float2 *__restrict__ tw, const Out &out)
{
    constexpr int G = 1 << LOG2G;
    const SmemOut in_place{s};
    stage<16, G, 1>(s, t, nullptr, tw, in_place);
    stage<16, G, 16>(s, t, tab, tw, in_place);
    if constexpr (LOG2G == 10) stage<4, G, 256>(s, t, tab + 64, tw, out);
    if constexpr (LOG2G == 11) stage<8, G, 256>(s, t, tab + 64, tw, out);
    if constexpr (LOG2G == 12) stage<16, G, 256>(s, t, tab + 64, tw, out);
    if constexpr (LOG2G >= 13) stage<16, G, 256>(s, t, tab + 64, tw, in_place);
    if constexpr (LOG2G == 13) stage<2, G, 4096>(s, t, nullptr, tw, out);
    if constexpr (LOG2G == 14) stage<4, G, 4096>(s, t, nullptr, tw, out);
}

}  // namespace fft
}  // namespace toi
