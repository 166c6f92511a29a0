// fft_smem.cuh -- power-of-two complex FFT of one sequence held in shared memory, the core of
// the pruned inverse transform of step a6 (k_fft.cu):
//   X[k] = sum_n x[n] exp(+2 pi i n k / G)        (unnormalised, sign +i: PAPER.md:301, DESIGN.md step 8)
// Decimation in frequency, IN PLACE, three stages of radices R1 = 16, R2, R3 (G = 16 R2 R3):
//   stage A  for b < G/16:            v[n1] = x[b + n1 G/16],        V = DFT16(v),   V[k1] *= W_G^(k1 b)
//   stage B  for k1, c < L/R2:        v[n2] = blk_k1[c + n2 L/R2],   V = DFT_R2(v),  V[k2] *= W_L^(k2 c)   (L = G/16)
//   stage C  for k1, k2:              v[n3] = blk_k1k2[n3],          V = DFT_R3(v)
// every butterfly writes back where it read, so a stage needs no barrier between its loads and its
// stores: ONE barrier per stage, a thread works through its butterflies one at a time (16 or 32
// elements in registers), and any number T of threads (G / 16 / T butterflies each) can share a
// sequence -- which is what lets G = 8192 and 16384 run with 256 / 512 threads.  Output k = k1 + 16 k2
// + 16 R2 k3 ends at position pos(k) = k1 G/16 + k2 R3 + k3 (digit-reversed); stage C hands
// its results to a functor out(k, address in place, value) in an order where consecutive threads hold
// consecutive k, so a pass can write them straight to global memory in natural order.
// Arithmetic: packed fp32 pairs (sm_100a FADD2 / FMUL2 / FFMA2: a complex add, or half a complex
// multiply, per instruction; the multiplication by +-i is an operand modifier).
// Padding: one element per 16, plus one per block of G/16 so that the block stride is odd:
// stage C's half-warp (16 different k1) then falls on 16 different bank pairs.
// Twiddles: W^m = exp(+2 pi i m / G) from a table of G float2 computed in fp64 on the host; per
// butterfly the powers w, w^2, w^4, w^8 (, w^16) of its base twiddle are looked up in per-stage tables
// in shared memory, the others are products of at most four of them.
#pragma once
#include <cuda_runtime.h>

namespace toi {
namespace fft {

typedef unsigned long long u64;

__device__ __forceinline__ u64 pk(float a, float b)
{
    u64 d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(a), "f"(b));
    return d;
}
__device__ __forceinline__ float2 up(u64 v)
{
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b)
{
    u64 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pk(a.x, a.y)), "l"(pk(b.x, b.y)));
    return up(d);
}
__device__ __forceinline__ float2 csub(float2 a, float2 b)
{
    u64 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pk(a.x, a.y)), "l"(pk(b.x, b.y)));
    return up(d);
}
__device__ __forceinline__ float2 muli(float2 a) { return make_float2(-a.y, a.x); }      // * (+i): folds into the consumer
// a w = a.x (w.x, w.y) + a.y (-w.y, w.x): FMUL2 + FFMA2
__device__ __forceinline__ float2 cmul(float2 a, float2 w)
{
    u64 t, r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(t) : "l"(pk(a.y, a.y)), "l"(pk(w.y, w.x)));
    const float2 tt = up(t);
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(pk(a.x, a.x)), "l"(pk(w.x, w.y)), "l"(pk(-tt.x, tt.y)));
    return up(r);
}

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
    v[3] = cmul(v[3], make_float2(h, h));
    v[5] = muli(v[5]);
    v[7] = cmul(v[7], make_float2(-h, h));
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

// first layer of a radix-32 butterfly (decimation in frequency): v[n] <- v[n] + v[n + 16] and
// v[n + 16] <- (v[n] - v[n + 16]) W32^n; DFT16 of the lower half then gives X[2 m], of the upper X[2 m + 1]
__device__ __forceinline__ void dft32_split(float2 *v)
{
    constexpr float kc[16] = {1.0f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                              0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f, 0.19509032201612826785f,
                              0.0f, -0.19509032201612826785f, -0.38268343236508977173f, -0.55557023301960222474f,
                              -0.70710678118654752440f, -0.83146961230254523708f, -0.92387953251128675613f, -0.98078528040323044913f};
    constexpr float ks[16] = {0.0f, 0.19509032201612826785f, 0.38268343236508977173f, 0.55557023301960222474f,
                              0.70710678118654752440f, 0.83146961230254523708f, 0.92387953251128675613f, 0.98078528040323044913f,
                              1.0f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                              0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f, 0.19509032201612826785f};
#pragma unroll
    for (int n = 0; n < 16; ++n) {
        const float2 d = csub(v[n], v[n + 16]);
        v[n] = cadd(v[n], v[n + 16]);
        v[n + 16] = n == 0 ? d : (n == 8 ? muli(d) : cmul(d, make_float2(kc[n], ks[n])));
    }
}

// v[r] *= w^r, r = 1 .. 15, from the powers p[0..3] = {w, w^2, w^4, w^8} of the butterfly's base twiddle
__device__ __forceinline__ void twiddle16(float2 *v, const float2 *p)
{
    const float2 w1 = p[0], w2 = p[1], w4 = p[2], w8 = p[3];
    const float2 w3 = cmul(w1, w2), w5 = cmul(w1, w4), w6 = cmul(w2, w4), w7 = cmul(w3, w4);
    v[1] = cmul(v[1], w1); v[2] = cmul(v[2], w2); v[3] = cmul(v[3], w3); v[4] = cmul(v[4], w4);
    v[5] = cmul(v[5], w5); v[6] = cmul(v[6], w6); v[7] = cmul(v[7], w7); v[8] = cmul(v[8], w8);
    v[9] = cmul(v[9], cmul(w1, w8)); v[10] = cmul(v[10], cmul(w2, w8)); v[11] = cmul(v[11], cmul(w3, w8));
    v[12] = cmul(v[12], cmul(w4, w8)); v[13] = cmul(v[13], cmul(w5, w8)); v[14] = cmul(v[14], cmul(w6, w8));
    v[15] = cmul(v[15], cmul(w7, w8));
}

// ---- shapes -------------------------------------------------------------------------------------
template <int LOG2G>
struct Plan {
    static_assert(LOG2G >= 10 && LOG2G <= 14, "G = 2^10 .. 2^14");
    static constexpr int G = 1 << LOG2G;
    static constexpr int R2 = LOG2G == 14 ? 32 : 16;
    static constexpr int R3 = G / (16 * R2);                 // 4, 8, 16, 32, 32
    static constexpr int L1 = G / 16;                        // block length after stage A
    static constexpr int S2 = L1 / R2;                       // stride of stage B = number of its base twiddles
    static constexpr int kDelta = 1;
    static constexpr int L1p = L1 + L1 / 16 + kDelta;        // padded block stride, odd
    static_assert(L1p % 2 == 1, "block stride must be odd");
    static constexpr int kPadded = 16 * L1p;                 // float2 per sequence
    static constexpr int kTabBWidth = R2 == 32 ? 8 : 4;      // powers stored per row of stage B's table
    static constexpr int kTabA = L1 * 4, kTabB = S2 * kTabBWidth;
    static constexpr int kTabFloat2 = kTabA + kTabB;
};

__device__ __forceinline__ int pad16(int e) { return e + (e >> 4); }

// where element i of the sequence sits
template <int LOG2G>
__device__ __forceinline__ int phys(int i)
{
    return i + (i >> 4) + (i >> (LOG2G - 4)) * Plan<LOG2G>::kDelta;
}
// where output k sits after an in-place stage C
template <int LOG2G>
__device__ __forceinline__ int phys_out(int k)
{
    using P = Plan<LOG2G>;
    constexpr int kLog2R2 = P::R2 == 32 ? 5 : 4;
    const int k1 = k & 15, k2 = (k >> 4) & (P::R2 - 1), k3 = k >> (4 + kLog2R2);
    return k1 * P::L1p + pad16(k2 * P::R3 + k3);
}

// Twiddle tables in shared memory, filled once per CTA from the global table W^m = exp(+2 pi i m / G):
//   A: row b < G/16:  {w, w^2, w^4, w^8},          w = W_G^b
//   B: row c < S2:    {w, w^2, w^4, w^8} (radix 32: {w^2, w^4, w^8, w^16, w}),  w = W_L1^c = W_G^(16 c)
template <int LOG2G>
__device__ __forceinline__ void fill_tables(float2 *tab, const float2 *__restrict__ tw, int tid, int n_threads)
{
    using P = Plan<LOG2G>;
    for (int e = tid; e < P::kTabA; e += n_threads) tab[e] = __ldg(tw + ((e >> 2) << (e & 3)));
    for (int e = tid; e < P::kTabB; e += n_threads) {
        const int c = e / P::kTabBWidth, q = e % P::kTabBWidth;
        const int sh = P::kTabBWidth == 8 ? (q < 4 ? q + 1 : 0) : q;        // radix 32: {w^2, w^4, w^8, w^16, w, -, -, -}
        tab[P::kTabA + e] = q < 5 ? __ldg(tw + (((16 * c) << sh) & (P::G - 1))) : make_float2(0.0f, 0.0f);
    }
}

struct SmemOut {        // stage C in place: the caller reads output k at phys_out(k) after a barrier
    __device__ __forceinline__ void operator()(int, float2 *at, float2 v) const { *at = v; }
};

__device__ __forceinline__ void load_powers(float2 *p, const float2 *row)
{
    const float4 lo = *reinterpret_cast<const float4 *>(row), hi = *reinterpret_cast<const float4 *>(row + 2);
    p[0] = make_float2(lo.x, lo.y); p[1] = make_float2(lo.z, lo.w);
    p[2] = make_float2(hi.x, hi.y); p[3] = make_float2(hi.z, hi.w);
}

// stage A: G/16 radix-16 butterflies of stride G/16, twiddled by W_G^(k1 b).  `in(b, r)` supplies element
// b + r G/16: from the sequence itself (SmemIn), or straight from global memory (consecutive threads,
// consecutive b), which saves the pass that would first park the sequence in shared memory.
struct SmemIn {
    const float2 *s;
    int l1p;
    __device__ __forceinline__ float2 operator()(int b, int r) const { return s[pad16(b) + r * l1p]; }
};

// one butterfly of stage A: loads through `in`, results to at[r L1p]
template <int LOG2G, class In>
__device__ __forceinline__ void stage_a_butterfly(float2 *at, int b, const float2 *tab, const In &in)
{
    using P = Plan<LOG2G>;
    float2 v[16], p[4];
#pragma unroll
    for (int r = 0; r < 16; ++r) v[r] = in(b, r);
    load_powers(p, tab + 4 * b);
    dft16(v);
    twiddle16(v, p);
#pragma unroll
    for (int r = 0; r < 16; ++r) at[r * P::L1p] = v[r];
}

template <int LOG2G, int T, class In>
__device__ __forceinline__ void stage_a(float2 *s, int t, const float2 *tab, const In &in)
{
    using P = Plan<LOG2G>;
    static_assert(P::L1 % T == 0, "threads per sequence must divide G / 16");
#pragma unroll 1
    for (int b = t; b < P::L1; b += T) stage_a_butterfly<LOG2G>(s + pad16(b), b, tab, in);
}

// stage B: inside block k1 (length L1), butterflies of radix R2 and stride S2, twiddled by W_L1^(k2 c)
template <int LOG2G, int T>
__device__ __forceinline__ void stage_b(float2 *s, int t, const float2 *tab)
{
    using P = Plan<LOG2G>;
    constexpr int NB = P::G / P::R2;
    static_assert(NB % T == 0, "threads per sequence must divide G / R2");
#pragma unroll 1
    for (int u = t; u < NB; u += T) {
        const int c = u % P::S2, k1 = u / P::S2;
        float2 *blk = s + k1 * P::L1p;
        if constexpr (P::R2 == 16) {
            float2 v[16], p[4];
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = blk[pad16(c + r * P::S2)];
            load_powers(p, tab + P::kTabA + 4 * c);
            dft16(v);
            twiddle16(v, p);
#pragma unroll
            for (int r = 0; r < 16; ++r) blk[pad16(c + r * P::S2)] = v[r];
        } else {
            // radix 32: X[2 m] = DFT16(lower)[m] (w^2)^m,  X[2 m + 1] = DFT16(upper)[m] (w^2)^m w
            float2 v[32], p[4];
#pragma unroll
            for (int r = 0; r < 32; ++r) v[r] = blk[pad16(c + r * P::S2)];
            const float2 *row = tab + P::kTabA + 8 * c;
            const float2 w1 = row[4];
            load_powers(p, row);
            dft32_split(v);
            dft16(v);
            twiddle16(v, p);
#pragma unroll
            for (int m = 0; m < 16; ++m) blk[pad16(c + 2 * m * P::S2)] = v[m];
            dft16(v + 16);
            twiddle16(v + 16, p);
#pragma unroll
            for (int m = 0; m < 16; ++m) blk[pad16(c + (2 * m + 1) * P::S2)] = cmul(v[16 + m], w1);
        }
    }
}

// stage C: the R3 contiguous elements of block (k1, k2), no twiddles; thread order tau = k1 + 16 k2 so that
// consecutive threads hold consecutive outputs k = tau + r (G / R3)
template <int LOG2G, int T, class Out>
__device__ __forceinline__ void stage_c(float2 *s, int t, const Out &out)
{
    using P = Plan<LOG2G>;
    constexpr int NB = P::G / P::R3;                     // = 16 R2
    static_assert(NB % T == 0, "threads per sequence must divide G / R3");
#pragma unroll 1
    for (int tau = t; tau < NB; tau += T) {
        const int k1 = tau & 15, k2 = tau >> 4;
        float2 *blk = s + k1 * P::L1p;
        const int e0 = k2 * P::R3;
        if constexpr (P::R3 == 32) {
            float2 v[32];
#pragma unroll
            for (int r = 0; r < 32; ++r) v[r] = blk[pad16(e0 + r)];
            dft32_split(v);
            dft16(v);
#pragma unroll
            for (int m = 0; m < 16; ++m) out(tau + 2 * m * NB, blk + pad16(e0 + 2 * m), v[m]);
            dft16(v + 16);
#pragma unroll
            for (int m = 0; m < 16; ++m) out(tau + (2 * m + 1) * NB, blk + pad16(e0 + 2 * m + 1), v[16 + m]);
        } else {
            float2 v[P::R3];
#pragma unroll
            for (int r = 0; r < P::R3; ++r) v[r] = blk[pad16(e0 + r)];
            if constexpr (P::R3 == 16) dft16(v);
            else if constexpr (P::R3 == 8) dft8(v);
            else dft4(v[0], v[1], v[2], v[3]);
#pragma unroll
            for (int r = 0; r < P::R3; ++r) out(tau + r * NB, blk + pad16(e0 + r), v[r]);
        }
    }
}

// The whole transform of the sequence at `s` (element i at phys<LOG2G>(i)), by T threads, t = my index
// among them.  Two CTA-wide barriers: every thread of the CTA must call it the same number of times;
// the caller puts a barrier between its stores of the sequence and this call, and after it.
// transform_from: stage A takes its inputs from `in` instead (the sequence need not be filled).
// `tab`: fill_tables' output.  Stage C's results go to `out`.
template <int LOG2G, int T, class In, class Out>
__device__ __forceinline__ void transform_from(float2 *s, int t, const float2 *tab, const In &in, const Out &out)
{
    stage_a<LOG2G, T>(s, t, tab, in);
    __syncthreads();
    stage_b<LOG2G, T>(s, t, tab);
    __syncthreads();
    stage_c<LOG2G, T>(s, t, out);
}
template <int LOG2G, int T, class Out>
__device__ __forceinline__ void transform(float2 *s, int t, const float2 *tab, const Out &out)
{
    transform_from<LOG2G, T>(s, t, tab, SmemIn{s, Plan<LOG2G>::L1p}, out);
}

}  // namespace fft
}  // namespace toi
