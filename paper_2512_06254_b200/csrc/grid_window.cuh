// grid_window.cuh -- the sliding register window shared by the gridding kernels (step a5):
//   grid[iv+dv][iu+du] += f z phi(iu+du-gu) phi(iv+dv-gv),  du, dv = -3..3
// 80-byte shared-memory records of pre-processed samples, the inline-PTX consume phase that
// accumulates them into an 8 x 8-cell window held in the registers of a group of 4 lanes (two
// column slots per lane, corner on even cells) and flushes retiring rows / columns with
// red.global.add.v2.f32, and the raw-input loads.  Design notes: DESIGN.md section 6.
#pragma once
#include "toi_internal.cuh"

namespace toi {
namespace {

constexpr int kGroups = 8;        // 4-lane groups per warp
constexpr int kBatch = 4;         // samples per group per pre-processing batch (8 * 4 = 32 lanes)
constexpr int kR = 8;             // rows (and column slots) of the register window
constexpr int kRecQuads = 5;      // record = 5 x 16 B: {zre, zim, wkey, pv0} {pv1..4} {pv5..7, 0} {pu0..3} {pu4..7}
constexpr int kGroupQuads = kBatch * kRecQuads;          // 20; group g sits at quad 20 g + (g >> 1):
constexpr int kWarpQuads = kGroups * kGroupQuads + 4;    // conflict-free STS.128 / LDS.128, spread tap words
constexpr unsigned kNoKey = 0x80008000u;   // (bv, bu) = (-32768, -32768): never a window base (G <= 32768)

constexpr int kHasW = 1, kHasF = 2, kHasD = 4;

__device__ __forceinline__ unsigned cell_key(int iu, int iv) { return ((unsigned)iv << 16) | ((unsigned)iu & 0xffffu); }
__device__ __forceinline__ int group_quad(int g) { return g * kGroupQuads + (g >> 1); }

// ---- the consume phase: one group of 4 lanes, 4 records ------------------------------------------
// Operands: %0..%7 rows of column set A, %8..%15 rows of set B, %16 tapA = window column my set A holds
// (0..7; set B holds tapA ^ 4), %17 ckey = packed base cell of the open window (kNoKey: closed),
// %18 / %19 = shared addresses of my A / B phi_u tap in record 0, %20 rgs = shared address of the
// group's records, %21 gc = &grid cell (0,0), %22 row stride in bytes, %23 G, %24 L = lane in group.
#define TOI8_HEAD(P, OFF)                                                                             \
    "ld.shared.v4.b32 {zx" #P ", zy" #P ", key" #P ", va" #P "}, [%20+" #OFF "];\n\t"                \
    "ld.shared.b32 pa" #P ", [%18+" #OFF "];\n\t"                                                     \
    "ld.shared.b32 pb" #P ", [%19+" #OFF "];\n\t"
#define TOI8_ROW(V, A, B)                                                                             \
    "mov.b64 bb, {" V ", " V "};\n\tfma.rn.f32x2 " A ", ta, bb, " A ";\n\tfma.rn.f32x2 " B ", tb, bb, " B ";\n\t"
#define TOI8_FMA(P)                                                                                   \
    "mov.b64 zz, {zx" #P ", zy" #P "};\n\t"                                                           \
    "mov.b64 bb, {pa" #P ", pa" #P "};\n\tmul.rn.f32x2 ta, zz, bb;\n\t"                               \
    "mov.b64 bb, {pb" #P ", pb" #P "};\n\tmul.rn.f32x2 tb, zz, bb;\n\t"                               \
    TOI8_ROW("va" #P, "%0", "%8") TOI8_ROW("v1", "%1", "%9") TOI8_ROW("v2", "%2", "%10")              \
    TOI8_ROW("v3", "%3", "%11") TOI8_ROW("v4", "%4", "%12") TOI8_ROW("v5", "%5", "%13")               \
    TOI8_ROW("v6", "%6", "%14") TOI8_ROW("v7", "%7", "%15")
#define TOI8_TEST(K, P, OFF16, OFF32)                                                                 \
    "ld.shared.v4.b32 {v1, v2, v3, v4}, [%20+" #OFF16 "];\n\t"                                        \
    "ld.shared.v4.b32 {v5, v6, v7, pad}, [%20+" #OFF32 "];\n\t"                                       \
    "setp.ne.u32 pq, key" #P ", %17;\n\t"                                                             \
    "@pq bra S" #K ";\n\t"                                                                            \
    "B" #K ":\n\t"
#define TOI8_REC(K, P, PN, OFF16, OFF32, OFFN) TOI8_TEST(K, P, OFF16, OFF32) TOI8_HEAD(PN, OFFN) TOI8_FMA(P)
#define TOI8_REC_LAST(K, P, OFF16, OFF32) TOI8_TEST(K, P, OFF16, OFF32) TOI8_FMA(P)

// q = &grid[row][col] from 32-bit row / col registers
#define TOI8_ADDR(ROW, COL)                                                                           \
    "mul.wide.s32 q, " ROW ", %23;\n\tcvt.s64.s32 q1, " COL ";\n\tadd.s64 q, q, q1;\n\t"             \
    "shl.b64 q, q, 3;\n\tadd.s64 q, %21, q;\n\t"
#define TOI8_RED(A) "mov.b64 {x, y}, " A ";\n\tred.global.add.v2.f32 [q], {x, y};\n\t"
// flush the 8 rows of one column set starting at q (row stride rs64) and clear them
#define TOI8_FLUSH8(A0, A1, A2, A3, A4, A5, A6, A7)                                                   \
    TOI8_RED(A0) "add.s64 q, q, rs64;\n\t" TOI8_RED(A1) "add.s64 q, q, rs64;\n\t"                     \
    TOI8_RED(A2) "add.s64 q, q, rs64;\n\t" TOI8_RED(A3) "add.s64 q, q, rs64;\n\t"                     \
    TOI8_RED(A4) "add.s64 q, q, rs64;\n\t" TOI8_RED(A5) "add.s64 q, q, rs64;\n\t"                     \
    TOI8_RED(A6) "add.s64 q, q, rs64;\n\t" TOI8_RED(A7)                                               \
    "@pz mov.b64 " A0 ", {pad, pad};\n\t@pz mov.b64 " A1 ", {pad, pad};\n\t@pz mov.b64 " A2 ", {pad, pad};\n\t" \
    "@pz mov.b64 " A3 ", {pad, pad};\n\t@pz mov.b64 " A4 ", {pad, pad};\n\t@pz mov.b64 " A5 ", {pad, pad};\n\t" \
    "@pz mov.b64 " A6 ", {pad, pad};\n\t@pz mov.b64 " A7 ", {pad, pad};\n\t"
#define TOI8_SHIFT_DOWN2(A0, A1, A2, A3, A4, A5, A6, A7)                                              \
    "@pz mul.rn.f32x2 " A0 ", " A2 ", one2;\n\t@pz mul.rn.f32x2 " A1 ", " A3 ", one2;\n\t"             \
    "@pz mul.rn.f32x2 " A2 ", " A4 ", one2;\n\t@pz mul.rn.f32x2 " A3 ", " A5 ", one2;\n\t"             \
    "@pz mul.rn.f32x2 " A4 ", " A6 ", one2;\n\t@pz mul.rn.f32x2 " A5 ", " A7 ", one2;\n\t"             \
    "@pz mov.b64 " A6 ", {pad, pad};\n\t@pz mov.b64 " A7 ", {pad, pad};\n\t"
#define TOI8_SHIFT_UP2(A0, A1, A2, A3, A4, A5, A6, A7)                                                \
    "@pz mul.rn.f32x2 " A7 ", " A5 ", one2;\n\t@pz mul.rn.f32x2 " A6 ", " A4 ", one2;\n\t"             \
    "@pz mul.rn.f32x2 " A5 ", " A3 ", one2;\n\t@pz mul.rn.f32x2 " A4 ", " A2 ", one2;\n\t"             \
    "@pz mul.rn.f32x2 " A3 ", " A1 ", one2;\n\t@pz mul.rn.f32x2 " A2 ", " A0 ", one2;\n\t"             \
    "@pz mov.b64 " A0 ", {pad, pad};\n\t@pz mov.b64 " A1 ", {pad, pad};\n\t"
#define TOI8_SETA "%0", "%1", "%2", "%3", "%4", "%5", "%6", "%7"
#define TOI8_SETB "%8", "%9", "%10", "%11", "%12", "%13", "%14", "%15"
#define TOI8_APPLY(M, ...) M(__VA_ARGS__)
// The window of my group moves to the base cell in key<P> (record K):
//   * "no sample" record (padding / off-grid): nothing moves;
//   * near move, (du, dv) each in {-2, 0, 2}: the lanes whose slots hold the two retiring columns
//     flush those sets (8 cells each) and the slots take the two entering columns; a row move
//     flushes two cells per set and shifts the rows by two registers;
//   * first sample of the strip, or a move by more than two cells: every set is flushed and the
//     window reopens at the new base.
// Addresses are formed on demand from the packed base cell (no per-lane column pointer is kept).
#define TOI8_SLOW(K, P, OFF)                                                                          \
    "S" #K ":\n\t"                                                                                    \
    "setp.eq.u32 pz, pad, 0;\n\t"                                                                     \
    "setp.eq.u32 p0, key" #P ", 0x80008000;\n\t"                                                      \
    "@p0 bra B" #K ";\n\t"                                                                            \
    "shl.b32 t1, key" #P ", 16;\n\tshr.s32 cu, t1, 16;\n\tshr.s32 cv, key" #P ", 16;\n\t"            \
    "shl.b32 t1, %17, 16;\n\tshr.s32 ou, t1, 16;\n\tshr.s32 ov, %17, 16;\n\t"                         \
    "sub.s32 du, cu, ou;\n\tsub.s32 dv, cv, ov;\n\t"                                                  \
    "add.s32 t1, du, 2;\n\tadd.s32 t2, dv, 2;\n\t"                                                    \
    "setp.ne.u32 po, %17, 0x80008000;\n\t"                /* window open */                           \
    "setp.le.and.u32 pn, t1, 4, po;\n\t"                                                              \
    "setp.le.and.u32 pn, t2, 4, pn;\n\t"                  /* near move */                             \
    "xor.b32 tpb, %16, 4;\n\t"                            /* window column of my set B */             \
    "setp.gt.s32 pu, du, 0;\n\t"                                                                      \
    "selp.s32 t1, 0, 3, pu;\n\t"                          /* retiring column pair: 0,1 or 6,7 */      \
    "setp.ne.and.s32 pc, du, 0, pn;\n\t"                                                              \
    "shr.u32 t2, %16, 1;\n\tsetp.eq.and.s32 pfa, t2, t1, pc;\n\t"                                     \
    "shr.u32 t2, tpb, 1;\n\tsetp.eq.and.s32 pfb, t2, t1, pc;\n\t"                                     \
    "not.pred pf, pn;\n\tand.pred pf, pf, po;\n\t"        /* far move of an open window: flush all */ \
    "or.pred pfa, pfa, pf;\n\tor.pred pfb, pfb, pf;\n\t"                                              \
    "cvt.u64.u32 rs64, %22;\n\t"                                                                      \
    "@!pfa bra NA" #K ";\n\t"                                                                         \
    "add.s32 t1, ou, %16;\n\t"                                                                        \
    TOI8_ADDR("ov", "t1")                                                                             \
    TOI8_APPLY(TOI8_FLUSH8, TOI8_SETA)                                                                \
    "NA" #K ":\n\t"                                                                                   \
    "@!pfb bra NB" #K ";\n\t"                                                                         \
    "add.s32 t1, ou, tpb;\n\t"                                                                        \
    TOI8_ADDR("ov", "t1")                                                                             \
    TOI8_APPLY(TOI8_FLUSH8, TOI8_SETB)                                                                \
    "NB" #K ":\n\t"                                                                                   \
    "@!pn bra O" #K ";\n\t"                                                                           \
    "sub.s32 t1, %16, du;\n\tand.b32 %16, t1, 7;\n\t"     /* my window columns after the column move */ \
    "xor.b32 tpb, %16, 4;\n\t"                                                                        \
    "setp.gt.s32 pu, dv, 0;\n\tsetp.lt.s32 pd, dv, 0;\n\t"                                            \
    "mov.b64 one2, 0x3f8000003f800000;\n\t"                                                           \
    "add.s32 t1, cu, %16;\n\t"                            /* my set-A column in the new window */     \
    "sub.s32 t2, tpb, %16;\n\tmul.wide.s32 q2, t2, 8;\n\t" /* set B sits 4 columns right or left */    \
    "@!pu bra NU" #K ";\n\t"                                                                          \
    TOI8_ADDR("ov", "t1")                                 /* dv = +2: rows ov, ov + 1 retire */       \
    TOI8_RED("%0") "add.s64 q, q, q2;\n\t" TOI8_RED("%8")                                             \
    "sub.s64 q, q, q2;\n\tadd.s64 q, q, rs64;\n\t"                                                    \
    TOI8_RED("%1") "add.s64 q, q, q2;\n\t" TOI8_RED("%9")                                             \
    TOI8_APPLY(TOI8_SHIFT_DOWN2, TOI8_SETA)                                                           \
    TOI8_APPLY(TOI8_SHIFT_DOWN2, TOI8_SETB)                                                           \
    "NU" #K ":\n\t"                                                                                   \
    "@!pd bra F" #K ";\n\t"                                                                           \
    "add.s32 t2, ov, 6;\n\t"                              /* dv = -2: rows ov + 6, ov + 7 retire */   \
    TOI8_ADDR("t2", "t1")                                                                             \
    TOI8_RED("%6") "add.s64 q, q, q2;\n\t" TOI8_RED("%14")                                            \
    "sub.s64 q, q, q2;\n\tadd.s64 q, q, rs64;\n\t"                                                    \
    TOI8_RED("%7") "add.s64 q, q, q2;\n\t" TOI8_RED("%15")                                            \
    TOI8_APPLY(TOI8_SHIFT_UP2, TOI8_SETA)                                                             \
    TOI8_APPLY(TOI8_SHIFT_UP2, TOI8_SETB)                                                             \
    "bra F" #K ";\n\t"                                                                                \
    "O" #K ":\n\t"                                                                                    \
    "sub.s32 t1, %24, cu;\n\tand.b32 %16, t1, 7;\n\t"     /* slot L holds window column (L - bu) mod 8 */ \
    "xor.b32 tpb, %16, 4;\n\t"                                                                        \
    "F" #K ":\n\t"                                                                                    \
    "mov.u32 %17, key" #P ";\n\t"                                                                     \
    "shl.b32 t1, %16, 2;\n\tadd.u32 t1, t1, 48;\n\tadd.u32 %18, %20, t1;\n\t"                         \
    "shl.b32 t1, tpb, 2;\n\tadd.u32 t1, t1, 48;\n\tadd.u32 %19, %20, t1;\n\t"                         \
    "ld.shared.b32 pa" #P ", [%18+" #OFF "];\n\t"                                                     \
    "ld.shared.b32 pb" #P ", [%19+" #OFF "];\n\t"                                                     \
    "bra B" #K ";\n\t"

__device__ __forceinline__ void consume_batch(u64 (&a)[kR], u64 (&b)[kR], unsigned &tapA, unsigned &ckey,
                                              unsigned &rpa, unsigned &rpb, unsigned rgs, const float2 *gc,
                                              unsigned rs, int G, int L)
{
    asm volatile(
        "{\n\t"
        ".reg .b32 zx0, zy0, key0, va0, pa0, pb0, zx1, zy1, key1, va1, pa1, pb1, pad, v1, v2, v3, v4, v5, v6, v7;\n\t"
        ".reg .b32 t1, t2, cu, cv, ou, ov, du, dv, tpb;\n\t"
        ".reg .b64 zz, ta, tb, bb, one2, q, q1, q2, rs64;\n\t"
        ".reg .f32 x, y;\n\t"
        ".reg .pred pq, p0, po, pn, pc, pf, pu, pd, pz, pfa, pfb;\n\t"
        TOI8_HEAD(0, 0)
        TOI8_REC(0, 0, 1, 16, 32, 80)
        TOI8_REC(1, 1, 0, 96, 112, 160)
        TOI8_REC(2, 0, 1, 176, 192, 240)
        TOI8_REC_LAST(3, 1, 256, 272)
        "bra DONE;\n\t"
        TOI8_SLOW(0, 0, 0)
        TOI8_SLOW(1, 1, 80)
        TOI8_SLOW(2, 0, 160)
        TOI8_SLOW(3, 1, 240)
        "DONE:\n\t"
        "}"
        : "+l"(a[0]), "+l"(a[1]), "+l"(a[2]), "+l"(a[3]), "+l"(a[4]), "+l"(a[5]), "+l"(a[6]), "+l"(a[7]),
          "+l"(b[0]), "+l"(b[1]), "+l"(b[2]), "+l"(b[3]), "+l"(b[4]), "+l"(b[5]), "+l"(b[6]), "+l"(b[7]),
          "+r"(tapA), "+r"(ckey), "+r"(rpa), "+r"(rpb)
        : "r"(rgs), "l"(gc), "r"(rs), "r"(G), "r"(L)
        : "memory");
}

// Strip end: flush the open window (base cell in ckey): my two column slots, 8 rows each.
__device__ __forceinline__ void flush_sets(const u64 (&a)[kR], const u64 (&b)[kR], unsigned tapA, unsigned ckey,
                                           const float2 *gc, long long rs, int G)
{
    const int ou = (int)(short)(ckey & 0xffffu), ov = (int)ckey >> 16;
#pragma unroll
    for (int set = 0; set < 2; ++set) {
        const unsigned tap = set ? (tapA ^ 4u) : tapA;
        const char *p = reinterpret_cast<const char *>(gc + ((long long)ov * G + (ou + (int)tap)));
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            const float2 v = unpack2(set ? b[r] : a[r]);
            asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" : : "l"(p), "f"(v.x), "f"(v.y) : "memory");
            p += rs;
        }
    }
}

// Raw inputs of one sample as they sit in HBM (requested one batch ahead; decoded at use).
struct Raw {
    float2 a, b;      // the two parallel hands
    float wa, wb;
    unsigned fl;      // raw flag bytes as loaded (layout depends on MODE); decoded at use
    double s;         // s_c = nu_c / c0 (not carried when the cell is computed a batch ahead)
};

// Geometry of one sample, computed one batch AHEAD of its data: the centre cell depends only on the
// baseline and the channel, so the dependent density lookup of uniform weighting (L2 latency under
// a streaming load: several hundred cycles) is in flight for a whole batch before it is needed.
struct Cell {
    unsigned key;     // packed BASE cell of the sample's window ((centre - 3) & ~1 per axis), kNoKey when off the grid
    unsigned sh;      // bit 0 / bit 1: the footprint starts at window column / row 1 instead of 0
    float xu, xv;     // sub-cell offsets
    float dens;       // D[cell] (1 when there is no density map or the sample is off the grid)
};

// MODE 4: n_p = 4, hands (0, 3), 16-B aligned weights and 4-B aligned flags -> 2 LDG.64 + LDG.128 + LDG.32
// MODE 2: n_p = 2, hands (0, 1), 8-B aligned weights, 2-B aligned flags     -> LDG.128 + LDG.64 + LDG.U16
// MODE 0: anything else, scalar loads
template <int MODE, bool WITH_S>
__device__ __forceinline__ void load_raw(const Geometry &g, const Inputs &in, bool has_w, bool has_f,
                                         long long q, int c, Raw &r)
{
    r.s = WITH_S ? __ldg(g.s + c) : 0.0;
    r.wa = r.wb = 1.0f;
    r.fl = 0u;
    if (MODE == 4) {
        const float2 *v = in.vis + 4 * q;
        r.a = __ldcs(v);
        r.b = __ldcs(v + 3);
        if (has_w) {
            const float4 w = __ldcs(reinterpret_cast<const float4 *>(in.weights) + q);
            r.wa = w.x; r.wb = w.w;
        }
        if (has_f) r.fl = __ldcs(reinterpret_cast<const unsigned *>(in.flags) + q);
    } else if (MODE == 2) {
        const float4 v = __ldcs(reinterpret_cast<const float4 *>(in.vis) + q);
        r.a = make_float2(v.x, v.y);
        r.b = make_float2(v.z, v.w);
        if (has_w) {
            const float2 w = __ldcs(reinterpret_cast<const float2 *>(in.weights) + q);
            r.wa = w.x; r.wb = w.y;
        }
        if (has_f) r.fl = __ldcs(reinterpret_cast<const unsigned short *>(in.flags) + q);
    } else {
        const long long o = q * g.n_p;
        r.a = __ldcs(in.vis + o + g.pol_a);
        r.b = __ldcs(in.vis + o + g.pol_b);
        if (has_w) { r.wa = __ldcs(in.weights + o + g.pol_a); r.wb = __ldcs(in.weights + o + g.pol_b); }
        if (has_f) r.fl = (unsigned)__ldcs(in.flags + o + g.pol_a) | ((unsigned)__ldcs(in.flags + o + g.pol_b) << 24);
        if (g.pol_b == g.pol_a) r.fl |= 0xff000000u;     // single hand: b never contributes
    }
}

}  // namespace
}  // namespace toi
