// k_grid_sliding.cu -- step a5, the product gridder (TOI_GRIDDER_SLIDING):
//   grid[iv+dv][iu+du] += f z phi(iu+du-gu) phi(iv+dv-gv),  du, dv = -3..3
// ("place visibilities on a grid"; kernel, support and edge rule: DESIGN.md G9, G10).
//
// Design (sm_100a; none of it is the paper's -- DESIGN.md section 6):
//  * The samples of one baseline lie on a ray through the uv origin, monotone in channel, and move
//    a few hundredths of a cell per channel: consecutive channels share a 7x7 footprint for many
//    samples and the footprint then slides by ONE cell.  So a group of 7 lanes keeps the whole
//    7x7 complex footprint in registers (lane = column, 7 row accumulators of packed re/im) and
//    streams through a strip of consecutive channels.  Per sample each lane issues one FMUL2
//    (z * phi_u[column]) and seven FFMA2 whose third operand is the scalar phi_v[row] broadcast
//    to both halves (the .F32 operand form of sm_100's FFMA2) -- 8 issue slots for 49 complex taps.
//  * When the centre cell moves by one column, only the retiring column (7 cells, one lane) is
//    flushed; the lane then owns the entering column (columns are owned by absolute column mod 7,
//    so nothing is shuffled).  When it moves by one row, the retiring row is flushed (one cell
//    per lane, 56 contiguous bytes) and the row accumulators shift by one register.  Flushes are
//    vector reductions red.global.add.v2.f32 (one per complex cell) onto the CENTRED grid, whose
//    addresses are affine in the cell (no wrap-around tests).  Per run of ~17 samples that is 7
//    reductions instead of 17 * 98 scalar atomics.
//  * A warp carries four such groups (28 of 32 lanes) on four adjacent strips of one baseline.
//    All 32 lanes first pre-process 32 samples (fp64 cell index, flags/weights/polarisation
//    average, 14 kernel taps as even/odd polynomials packed for both axes) into
//    an 80-byte shared-memory record each; the groups then consume their 8 records.  The consume
//    phase is ONE inline-PTX block: the eight record bodies are straight-line code with
//    immediate-offset LDS (next record's header prefetched), each with its own out-of-line
//    window-move block, and the accumulators never leave their register pairs.
//    The raw inputs of the next batch are requested before the current one is processed (register
//    prefetch), so HBM latency overlaps a whole batch of arithmetic.  Tasks (baseline, block of
//    4 strips) come from an atomic queue; the grid is persistent.
//  * fp32 summation is blocked by construction: register chains are bounded by the time a cell
//    stays inside a sliding window (tens to a few hundred samples), everything else is summed by
//    the L2 reduction units.
#include <stdlib.h>

#include "toi_internal.cuh"

namespace toi {
namespace {

constexpr int kGroups = 4;        // 7-lane groups per warp
constexpr int kBatch = 8;         // samples per group per pre-processing batch (4 * 8 = 32 lanes)
constexpr int kWarps = 8;         // warps per CTA
constexpr int kCtasPerSm = 3;     // resident CTAs per SM (80 registers per thread; 4 x 64 measured slower)
constexpr int kRecQuads = 5;      // record = 5 x 16 B: {zre, zim, key, pv0} {pv1..4} {pv5, pv6, 0, 0} {pu0..3} {pu4..6, 0}
constexpr int kGroupQuads = kBatch * kRecQuads + 2;   // +32 B: groups land on distinct banks
constexpr int kWarpQuads = kGroups * kGroupQuads;
constexpr unsigned kNoKey = 0x80008000u;   // (iv, iu) = (-32768, -32768): never an on-grid cell

// option bits of the kernel template: what is known at compile time about the optional inputs
constexpr int kHasW = 1, kHasF = 2, kHasD = 4;

// centre cell packed into one word: one compare per sample decides "same footprint as before"
__device__ __forceinline__ unsigned cell_key(int iu, int iv) { return ((unsigned)iv << 16) | ((unsigned)iu & 0xffffu); }

// Flush one window column (7 rows, row stride rs bytes, first row at p).  One asm block: the
// accumulators stay in their register pairs and the address walks by one 64-bit add.
__device__ __forceinline__ void flush_col(const u64 (&a)[kW], const char *p, long long rs)
{
    asm volatile(
        "{\n\t.reg .u64 p;\n\t.reg .f32 x, y;\n\t"
        "mov.u64 p, %7;\n\t"
        "mov.b64 {x, y}, %0;\n\tred.global.add.v2.f32 [p], {x, y};\n\tadd.s64 p, p, %8;\n\t"
        "mov.b64 {x, y}, %1;\n\tred.global.add.v2.f32 [p], {x, y};\n\tadd.s64 p, p, %8;\n\t"
        "mov.b64 {x, y}, %2;\n\tred.global.add.v2.f32 [p], {x, y};\n\tadd.s64 p, p, %8;\n\t"
        "mov.b64 {x, y}, %3;\n\tred.global.add.v2.f32 [p], {x, y};\n\tadd.s64 p, p, %8;\n\t"
        "mov.b64 {x, y}, %4;\n\tred.global.add.v2.f32 [p], {x, y};\n\tadd.s64 p, p, %8;\n\t"
        "mov.b64 {x, y}, %5;\n\tred.global.add.v2.f32 [p], {x, y};\n\tadd.s64 p, p, %8;\n\t"
        "mov.b64 {x, y}, %6;\n\tred.global.add.v2.f32 [p], {x, y};\n\t}"
        :
        : "l"(a[0]), "l"(a[1]), "l"(a[2]), "l"(a[3]), "l"(a[4]), "l"(a[5]), "l"(a[6]), "l"(p), "l"(rs)
        : "memory");
}

// ---- the consume phase: one group of 7 lanes, 8 records ------------------------------------------
// Operands: %0..%6 acc rows, %7 pcol = &grid[cv-3][my column], %8 mydu = which tap column this lane
// holds, %9 ckey = packed centre cell of the open window (kNoKey: closed), %10 rpu = shared address
// of my phi_u tap in record 0, %11 rgs = shared address of the group's records, %12 gc = &grid
// cell (0,0), %13 row stride in bytes (32-bit), %14 G, %15 m = this lane's column residue.
//
// Record k (parity P = k & 1 names the header registers): the header {z, key} and my phi_u tap were
// prefetched by record k-1; load the phi_v row, compare the key; the fast path is 4 LDS (2 of them
// the next header), 1 FMUL2, 7 FFMA2, 1 compare, 1 branch.  A changed key leaves to the record's
// own out-of-line block S<k> (an if-then diamond that reconverges at B<k>, so the four groups of
// a warp are split only while one of them moves its window), which slides or reopens the window
// and reloads my phi_u tap.
#define TOI_REC_HEAD(P, OFF)                                                                          \
    "ld.shared.v4.b32 {zx" #P ", zy" #P ", key" #P ", va" #P "}, [%11+" #OFF "];\n\t"                \
    "ld.shared.b32 pw" #P ", [%10+" #OFF "];\n\t"
#define TOI_REC_FMA(P)                                                                                \
    "mov.b64 tt, {zx" #P ", zy" #P "};\n\tmov.b64 bb, {pw" #P ", pw" #P "};\n\t"                     \
    "mul.rn.f32x2 tt, tt, bb;\n\t"                                                                    \
    "mov.b64 bb, {va" #P ", va" #P "};\n\tfma.rn.f32x2 %0, tt, bb, %0;\n\t"                          \
    "mov.b64 bb, {v1, v1};\n\tfma.rn.f32x2 %1, tt, bb, %1;\n\t"                                       \
    "mov.b64 bb, {v2, v2};\n\tfma.rn.f32x2 %2, tt, bb, %2;\n\t"                                       \
    "mov.b64 bb, {v3, v3};\n\tfma.rn.f32x2 %3, tt, bb, %3;\n\t"                                       \
    "mov.b64 bb, {v4, v4};\n\tfma.rn.f32x2 %4, tt, bb, %4;\n\t"                                       \
    "mov.b64 bb, {v5, v5};\n\tfma.rn.f32x2 %5, tt, bb, %5;\n\t"                                       \
    "mov.b64 bb, {v6, v6};\n\tfma.rn.f32x2 %6, tt, bb, %6;\n\t"
#define TOI_REC_TEST(K, P, OFF16, OFF32)                                                              \
    "ld.shared.v4.b32 {v1, v2, v3, v4}, [%11+" #OFF16 "];\n\t"                                        \
    "ld.shared.v2.b32 {v5, v6}, [%11+" #OFF32 "];\n\t"                                                \
    "setp.ne.u32 pq, key" #P ", %9;\n\t"                                                              \
    "@pq bra S" #K ";\n\t"                                                                            \
    "B" #K ":\n\t"
#define TOI_REC(K, P, PN, OFF16, OFF32, OFFN)                                                         \
    TOI_REC_TEST(K, P, OFF16, OFF32) TOI_REC_HEAD(PN, OFFN) TOI_REC_FMA(P)
#define TOI_REC_LAST(K, P, OFF16, OFF32) TOI_REC_TEST(K, P, OFF16, OFF32) TOI_REC_FMA(P)
#define TOI_FLUSH7(A0, A1, A2, A3, A4, A5, A6)                                                        \
    "mov.u64 q, %7;\n\tcvt.u64.u32 q1, %13;\n\t"                                                     \
    "mov.b64 {x, y}, " A0 ";\n\tred.global.add.v2.f32 [q], {x, y};\n\tadd.s64 q, q, q1;\n\t"          \
    "mov.b64 {x, y}, " A1 ";\n\tred.global.add.v2.f32 [q], {x, y};\n\tadd.s64 q, q, q1;\n\t"          \
    "mov.b64 {x, y}, " A2 ";\n\tred.global.add.v2.f32 [q], {x, y};\n\tadd.s64 q, q, q1;\n\t"          \
    "mov.b64 {x, y}, " A3 ";\n\tred.global.add.v2.f32 [q], {x, y};\n\tadd.s64 q, q, q1;\n\t"          \
    "mov.b64 {x, y}, " A4 ";\n\tred.global.add.v2.f32 [q], {x, y};\n\tadd.s64 q, q, q1;\n\t"          \
    "mov.b64 {x, y}, " A5 ";\n\tred.global.add.v2.f32 [q], {x, y};\n\tadd.s64 q, q, q1;\n\t"          \
    "mov.b64 {x, y}, " A6 ";\n\tred.global.add.v2.f32 [q], {x, y};\n\t"                               \
    "@pz mov.b64 " A0 ", {pad, pad};\n\t@pz mov.b64 " A1 ", {pad, pad};\n\t@pz mov.b64 " A2 ", {pad, pad};\n\t"   \
    "@pz mov.b64 " A3 ", {pad, pad};\n\t@pz mov.b64 " A4 ", {pad, pad};\n\t@pz mov.b64 " A5 ", {pad, pad};\n\t"   \
    "@pz mov.b64 " A6 ", {pad, pad};\n\t"
// The window of my group moves to the cell in key<P> (record K):
//   * "no sample" record (padding / off-grid): nothing moves;
//   * near move, (du, dv) each in {-1, 0, 1}: the lane that holds the retiring column flushes its 7
//     cells and takes over the entering column; a row move flushes one cell per lane and shifts the
//     row accumulators by one register;
//   * first sample of the strip, or a move by more than one cell: every lane flushes its column
//     (if the window was open) and the window reopens at (cu, cv).
// Flushes are red.global.add.v2.f32; freed accumulators are cleared from `pad`, an always-zero
// word of the records read once per batch (an immediate zero makes ptxas stage it through uniform
// registers).
// EVERY write to an accumulator in these blocks is predicated on pz = (pad == 0), which is always
// true but opaque to ptxas: a predicated write must leave the old value in place when the predicate
// is false, so the accumulator cannot be renamed across the block.  With plain writes ptxas joined
// the fast path to the block's register assignment by 10 MOVs per record (24 -> 13 instructions
// per record body once they are gone).
#define TOI_SLOW(K, P, OFF)                                                                           \
    "S" #K ":\n\t"                                                                                    \
    "setp.eq.u32 pz, pad, 0;\n\t"                                                                     \
    "setp.eq.u32 p0, key" #P ", 0x80008000;\n\t"                                                      \
    "@p0 bra B" #K ";\n\t"                                                                            \
    "shl.b32 t1, key" #P ", 16;\n\tshr.s32 cu, t1, 16;\n\tshr.s32 cv, key" #P ", 16;\n\t"            \
    "shl.b32 t1, %9, 16;\n\tshr.s32 ou, t1, 16;\n\tshr.s32 ov, %9, 16;\n\t"                           \
    "sub.s32 du, cu, ou;\n\tsub.s32 dv, cv, ov;\n\t"                                                  \
    "add.s32 t1, du, 1;\n\tadd.s32 t2, dv, 1;\n\t"                                                    \
    "setp.ne.u32 po, %9, 0x80008000;\n\t"                 /* window open */                           \
    "setp.le.and.u32 pn, t1, 2, po;\n\t"                                                              \
    "setp.le.and.u32 pn, t2, 2, pn;\n\t"                  /* near move */                             \
    "setp.gt.s32 pu, du, 0;\n\t"                                                                      \
    "selp.s32 t1, 0, 6, pu;\n\t"                                                                      \
    "setp.ne.and.s32 pc, du, 0, pn;\n\t"                                                              \
    "setp.eq.and.s32 pc, %8, t1, pc;\n\t"                 /* I hold the retiring column */            \
    "not.pred pf, pn;\n\t"                                                                            \
    "and.pred pf, pf, po;\n\t"                                                                        \
    "or.pred pf, pf, pc;\n\t"                             /* flush my column */                       \
    "@!pf bra NF" #K ";\n\t"                                                                          \
    TOI_FLUSH7("%0", "%1", "%2", "%3", "%4", "%5", "%6")                                              \
    "NF" #K ":\n\t"                                                                                   \
    "@!pn bra O" #K ";\n\t"                                                                           \
    "@pc mad.wide.s32 %7, du, 56, %7;\n\t"                                                            \
    "@pc mad.lo.s32 %8, du, 7, %8;\n\t"                                                               \
    "sub.s32 %8, %8, du;\n\t"                                                                         \
    "setp.gt.s32 pu, dv, 0;\n\t"                                                                      \
    "setp.lt.s32 pd, dv, 0;\n\t"                                                                      \
    "mov.b64 one2, 0x3f8000003f800000;\n\t"            /* rows shift by x * 1 (exact), one FMUL2   */ \
                                                        /* per row: a plain mov would be coalesced  */ \
                                                        /* away here and paid for on the fast path  */ \
    "@!pu bra NU" #K ";\n\t"                                                                          \
    "mov.b64 {x, y}, %0;\n\t"                                                                         \
    "red.global.add.v2.f32 [%7], {x, y};\n\t"                                                         \
    "@pz mul.rn.f32x2 %0, %1, one2;\n\t@pz mul.rn.f32x2 %1, %2, one2;\n\t@pz mul.rn.f32x2 %2, %3, one2;\n\t"      \
    "@pz mul.rn.f32x2 %3, %4, one2;\n\t@pz mul.rn.f32x2 %4, %5, one2;\n\t@pz mul.rn.f32x2 %5, %6, one2;\n\t"      \
    "@pz mov.b64 %6, {pad, pad};\n\t"                                                                   \
    "mad.wide.u32 %7, %13, 1, %7;\n\t"                                                                \
    "NU" #K ":\n\t"                                                                                   \
    "@!pd bra F" #K ";\n\t"                                                                           \
    "mad.wide.u32 q, %13, 6, %7;\n\t"                                                                 \
    "mov.b64 {x, y}, %6;\n\t"                                                                         \
    "red.global.add.v2.f32 [q], {x, y};\n\t"                                                          \
    "@pz mul.rn.f32x2 %6, %5, one2;\n\t@pz mul.rn.f32x2 %5, %4, one2;\n\t@pz mul.rn.f32x2 %4, %3, one2;\n\t"      \
    "@pz mul.rn.f32x2 %3, %2, one2;\n\t@pz mul.rn.f32x2 %2, %1, one2;\n\t@pz mul.rn.f32x2 %1, %0, one2;\n\t"      \
    "@pz mov.b64 %0, {pad, pad};\n\t"                                                                   \
    "cvt.u64.u32 q1, %13;\n\tsub.s64 %7, %7, q1;\n\t"                                                 \
    "bra F" #K ";\n\t"                                                                                \
    "O" #K ":\n\t"                                                                                    \
    "sub.s32 t1, %15, cu;\n\t"                                                                        \
    "add.s32 t1, t1, 7340035;\n\t"                        /* + 3 + (7 << 20): a true mod below */     \
    "mul.hi.u32 t2, t1, 2454267027;\n\tshr.u32 t2, t2, 2;\n\t" /* t1 / 7, exact below 2^31 */         \
    "mad.lo.s32 %8, t2, -7, t1;\n\t"                      /* column (cu - 3 + mydu) = m (mod 7) */    \
    "sub.s32 t2, cv, 3;\n\t"                                                                          \
    "mul.wide.s32 q, t2, %14;\n\t"                                                                    \
    "add.s32 t1, cu, %8;\n\t"                                                                         \
    "sub.s32 t1, t1, 3;\n\t"                                                                          \
    "cvt.s64.s32 q1, t1;\n\t"                                                                         \
    "add.s64 q, q, q1;\n\t"                                                                           \
    "shl.b64 q, q, 3;\n\t"                                                                            \
    "add.s64 %7, %12, q;\n\t"                                                                         \
    "F" #K ":\n\t"                                                                                    \
    "mov.u32 %9, key" #P ";\n\t"                                                                      \
    "shl.b32 t1, %8, 2;\n\t"                                                                          \
    "add.u32 t1, t1, 48;\n\t"                                                                         \
    "add.u32 %10, %11, t1;\n\t"                                                                       \
    "ld.shared.b32 pw" #P ", [%10+" #OFF "];\n\t"                                                     \
    "bra B" #K ";\n\t"

__device__ __forceinline__ void consume_batch(u64 (&a)[kW], const char *&pcol, int &mydu, unsigned &ckey,
                                              unsigned &rpu, unsigned rgs, const float2 *gc, long long rs,
                                              int G, int m)
{
    asm volatile(
        "{\n\t"
        ".reg .b32 zx0, zy0, key0, va0, pw0, zx1, zy1, key1, va1, pw1, pad, v1, v2, v3, v4, v5, v6;\n\t"
        ".reg .b32 t1, t2, cu, cv, ou, ov, du, dv;\n\t"
        ".reg .b64 tt, bb, one2, q, q1;\n\t"
        ".reg .f32 x, y;\n\t"
        ".reg .pred pq, p0, po, pn, pc, pf, pu, pd, pz;\n\t"
        "ld.shared.b32 pad, [%11+40];\n\t"      /* the always-zero third word of a record's third quad */
        TOI_REC_HEAD(0, 0)
        TOI_REC(0, 0, 1, 16, 32, 80)
        TOI_REC(1, 1, 0, 96, 112, 160)
        TOI_REC(2, 0, 1, 176, 192, 240)
        TOI_REC(3, 1, 0, 256, 272, 320)
        TOI_REC(4, 0, 1, 336, 352, 400)
        TOI_REC(5, 1, 0, 416, 432, 480)
        TOI_REC(6, 0, 1, 496, 512, 560)
        TOI_REC_LAST(7, 1, 576, 592)
        "bra DONE;\n\t"
        // ---------------- out of line: one window-move block per record ----------------
        TOI_SLOW(0, 0, 0)
        TOI_SLOW(1, 1, 80)
        TOI_SLOW(2, 0, 160)
        TOI_SLOW(3, 1, 240)
        TOI_SLOW(4, 0, 320)
        TOI_SLOW(5, 1, 400)
        TOI_SLOW(6, 0, 480)
        TOI_SLOW(7, 1, 560)
        "DONE:\n\t"
        "}"
        : "+l"(a[0]), "+l"(a[1]), "+l"(a[2]), "+l"(a[3]), "+l"(a[4]), "+l"(a[5]), "+l"(a[6]),
          "+l"(pcol), "+r"(mydu), "+r"(ckey), "+r"(rpu)
        : "r"(rgs), "l"(gc), "r"((unsigned)rs), "r"(G), "r"(m)
        : "memory");
}

// Raw inputs of one sample as they sit in HBM (requested one batch ahead; decoded at use, so the
// request really is a prefetch).
struct Raw {
    float2 a, b;      // the two parallel hands
    float wa, wb;
    unsigned fl;      // raw flag bytes as loaded (layout depends on MODE); decoded at use
    double s;         // s_c = nu_c / c0
};

// MODE 4: n_p = 4, hands (0, 3), 16-B aligned weights and 4-B aligned flags -> 2 LDG.64 + LDG.128 + LDG.32
// MODE 2: n_p = 2, hands (0, 1), 8-B aligned weights, 2-B aligned flags     -> LDG.128 + LDG.64 + LDG.U16
// MODE 0: anything else, scalar loads
// The raw inputs are read exactly once: __ldcs (evict-first) keeps them from displacing the density
// lines and the channel-scale table, which ARE re-read, from L1/L2.
template <int MODE>
__device__ __forceinline__ void load_raw(const Geometry &g, const Inputs &in, bool has_w, bool has_f,
                                         long long q, int c, Raw &r)
{
    r.s = __ldg(g.s + c);
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

// OPT >= 0: bits kHasW | kHasF | kHasD say at compile time which optional inputs exist;
// OPT < 0: decided at run time from the pointers.
template <int MODE, int OPT>
__global__ void __launch_bounds__(kWarps * 32, kCtasPerSm)
k_grid_sliding(Geometry g, Inputs in, SnapState *__restrict__ st, const float *__restrict__ D,
               float2 *__restrict__ grid, int strip_len, int tasks_per_row, unsigned n_tasks)
{
    __shared__ uint4 s_rec[kWarps * kWarpQuads];
    if (st->status != TOI_OK) return;
    const bool has_w = OPT >= 0 ? (OPT & kHasW) != 0 : in.weights != nullptr;
    const bool has_f = OPT >= 0 ? (OPT & kHasF) != 0 : in.flags != nullptr;
    const bool has_d = OPT >= 0 ? (OPT & kHasD) != 0 : D != nullptr;
    const int lane = threadIdx.x & 31;
    uint4 *rec = s_rec + (threadIdx.x >> 5) * kWarpQuads;

    // roles: every lane pre-processes one sample per batch (strip pre_g, channel pre_k of the
    // batch: 8 consecutive samples per strip = 256 contiguous bytes of visibilities); lanes 0..27
    // accumulate (group grp = strip, lane m of the group = one column of the footprint)
    const int pre_g = lane >> 3, pre_k = lane & 7;
    uint4 *my_rec = rec + pre_g * kGroupQuads + pre_k * kRecQuads;
    const bool acc_lane = lane < 7 * kGroups;
    const int grp = acc_lane ? lane / 7 : 0, m = lane - 7 * grp;
    const unsigned rgs = (unsigned)__cvta_generic_to_shared(rec + grp * kGroupQuads);
    const int G = g.G;
    const float2 *const gc = grid + centre_index(0, 0, G);   // cell (0, 0)
    const long long rs = (long long)G * 8;                   // row stride in bytes
    const float *const Dc = has_d ? D + centre_index(0, 0, G) : nullptr;

    double wsum = 0.0;
    unsigned n_grid = 0, n_off = 0, n_flag = 0;

    for (;;) {
        unsigned task = 0;
        if (lane == 0) task = atomicAdd(&st->task_counter, 1u);
        task = __shfl_sync(0xffffffffu, task, 0);
        if (task >= n_tasks) break;
        const int j = (int)(task / (unsigned)tasks_per_row);
        const int c_task = (int)(task % (unsigned)tasks_per_row) * (kGroups * strip_len);
        double rho1, rho2;
        rotate_baseline(st->V, in.uvw + 3 * j, rho1, rho2);
        const int c_lo = c_task + pre_g * strip_len + pre_k;      // my channel in batch 0
        const int c_hi = min(c_task + (pre_g + 1) * strip_len, g.n_c);
        const long long q_row = (long long)j * g.n_c;

        // sliding-window state of my group (uniform across its 7 lanes)
        u64 acc[kW];
#pragma unroll
        for (int d = 0; d < kW; ++d) acc[d] = 0ull;
        unsigned ckey = kNoKey;              // closed window; else the packed centre cell (cu, cv)
        int mydu = 0;                        // which tap column of the window this lane holds
        const char *pcol = nullptr;          // &grid[cv - 3][cu - 3 + mydu]: top of my column
        unsigned rpu = rgs + 48;             // shared address of my phi_u tap in record 0
        float wpart = 0.0f;

        Raw nxt;
        nxt.a = nxt.b = make_float2(0.0f, 0.0f); nxt.wa = nxt.wb = 0.0f; nxt.fl = 0u; nxt.s = 0.0;
        if (c_lo < c_hi) load_raw<MODE>(g, in, has_w, has_f, q_row + c_lo, c_lo, nxt);

        for (int b = 0; b < strip_len && c_task + b < g.n_c; b += kBatch) {
            // ---------------- pre-process one sample per lane ----------------
            {
                const int c = c_lo + b;
                const Raw cur = nxt;
                if (c + kBatch < c_hi && b + kBatch < strip_len)
                    load_raw<MODE>(g, in, has_w, has_f, q_row + c + kBatch, c + kBatch, nxt);
                unsigned key = kNoKey;
                bool valid = false;
                float wI = 0.0f, zx = 0.0f, zy = 0.0f, dens = 1.0f, pv0 = 0.0f;
                if (c < c_hi) {
                    int iu, iv;
                    float xu, xv;
                    sample_cell(rho1, rho2, cur.s, g.kappa, iu, iv, xu, xv);
                    if (!cell_on_grid(iu, iv, G)) {
                        ++n_off;
                    } else {
                        // a flagged sample keeps its own cell as key (z = 0, zero taps): it moves the
                        // window exactly as its unflagged neighbours do and never takes the slow path
                        key = cell_key(iu, iv);
                        // flag bytes of the two hands inside the raw word (decoded here, not at the load)
                        constexpr unsigned fmask_b = MODE == 2 ? 0x0000ff00u : 0xff000000u;
                        const float wa = (weight_ok(cur.wa) && !(cur.fl & 0x000000ffu)) ? cur.wa : 0.0f;
                        const float wb = (weight_ok(cur.wb) && !(cur.fl & fmask_b)) ? cur.wb : 0.0f;
                        wI = wa + wb;
                        if (!(wI > 0.0f)) {
                            ++n_flag;
                        } else {
                            ++n_grid;
                            valid = true;
                            if (has_d) dens = __ldg(Dc + ((long long)iv * G + iu));   // consumed last
                            // z = w_a Vis_a + w_b Vis_b; a zero-weight hand is skipped (its data may be NaN)
                            if (wa > 0.0f) { zx = wa * cur.a.x; zy = wa * cur.a.y; }
                            if (wb > 0.0f) { zx = fmaf(wb, cur.b.x, zx); zy = fmaf(wb, cur.b.y, zy); }
                            float pu[kW], pv[kW];
                            kernel_taps2(xu, xv, pu, pv);
                            pv0 = pv[0];
                            my_rec[1] = make_uint4(__float_as_uint(pv[1]), __float_as_uint(pv[2]), __float_as_uint(pv[3]), __float_as_uint(pv[4]));
                            my_rec[2] = make_uint4(__float_as_uint(pv[5]), __float_as_uint(pv[6]), 0u, 0u);
                            my_rec[3] = make_uint4(__float_as_uint(pu[0]), __float_as_uint(pu[1]), __float_as_uint(pu[2]), __float_as_uint(pu[3]));
                            my_rec[4] = make_uint4(__float_as_uint(pu[4]), __float_as_uint(pu[5]), __float_as_uint(pu[6]), 0u);
                        }
                    }
                }
                if (!valid) {
                    const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
                    my_rec[1] = zero; my_rec[2] = zero; my_rec[3] = zero; my_rec[4] = zero;
                }
                float f = 1.0f;
                if (has_d) asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(f) : "f"(dens));
                wpart = fmaf(f, wI, wpart);
                my_rec[0] = make_uint4(__float_as_uint(zx * f), __float_as_uint(zy * f), key, __float_as_uint(pv0));
            }
            __syncwarp();
            // ---------------- accumulate: group grp consumes its 8 records ----------------
            if (acc_lane) consume_batch(acc, pcol, mydu, ckey, rpu, rgs, gc, rs, G, m);
            __syncwarp();
        }
        // strip done: flush what is left of the window
        if (acc_lane && ckey != kNoKey) flush_col(acc, pcol, rs);
        wsum += (double)wpart;
    }

#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        wsum += __shfl_xor_sync(0xffffffffu, wsum, d);
        n_grid += __shfl_xor_sync(0xffffffffu, n_grid, d);
        n_off += __shfl_xor_sync(0xffffffffu, n_off, d);
        n_flag += __shfl_xor_sync(0xffffffffu, n_flag, d);
    }
    if (lane == 0) {
        if (wsum != 0.0) atomicAdd(&st->wsum, wsum);
        if (n_grid) atomicAdd(&st->n_gridded, (unsigned long long)n_grid);
        if (n_off) atomicAdd(&st->n_off_grid, (unsigned long long)n_off);
        if (n_flag) atomicAdd(&st->n_flagged, (unsigned long long)n_flag);
    }
}

template <int MODE>
void launch_mode(int opt, dim3 grid, dim3 block, cudaStream_t stream, const Geometry &g, const Inputs &in,
                 SnapState *st, const float *D, float2 *d_grid, int strip, int tasks_per_row, unsigned n_tasks)
{
#define TOI_LAUNCH(O) k_grid_sliding<MODE, O><<<grid, block, 0, stream>>>(g, in, st, D, d_grid, strip, tasks_per_row, n_tasks)
    switch (opt) {
    case kHasW | kHasF | kHasD: TOI_LAUNCH(kHasW | kHasF | kHasD); break;
    case kHasW | kHasF: TOI_LAUNCH(kHasW | kHasF); break;
    case kHasD: TOI_LAUNCH(kHasD); break;
    case 0: TOI_LAUNCH(0); break;
    default: TOI_LAUNCH(-1); break;
    }
#undef TOI_LAUNCH
}

}  // namespace

void launch_grid_sliding(const Geometry &g, const Inputs &in, SnapState *st, const float *d_density,
                         float2 *d_grid, int n_sms, cudaStream_t stream)
{
    // strip length (channels per group per task): long strips amortise the 49-cell flush at a strip
    // end, short ones balance the persistent grid's tail.  Aim at >= 6 tasks per resident warp,
    // within [32, 256] channels and a multiple of the 8-sample batch.
    const long long warps = (long long)kCtasPerSm * n_sms * kWarps;
    const long long want = ((long long)g.n_b * g.n_c) / (kGroups * 6 * warps);
    int strip = pick_strip(g.n_c, kGroups, kBatch, want, 32, 256);
    if (const char *e = getenv("TOI_STRIP")) strip = atoi(e);   // tuning override (multiple of 8)
    const int tasks_per_row = (g.n_c + kGroups * strip - 1) / (kGroups * strip);
    const long long n_tasks = (long long)g.n_b * tasks_per_row;
    long long ctas = (n_tasks + kWarps - 1) / kWarps;
    if (ctas > (long long)kCtasPerSm * n_sms) ctas = (long long)kCtasPerSm * n_sms;   // persistent CTAs pull from the queue
    const dim3 grid((unsigned)ctas), block(kWarps * 32);
    const uintptr_t aw = (uintptr_t)in.weights, af = (uintptr_t)in.flags, av = (uintptr_t)in.vis;
    const int opt = (in.weights ? kHasW : 0) | (in.flags ? kHasF : 0) | (d_density ? kHasD : 0);
    if (g.n_p == 4 && g.pol_a == 0 && g.pol_b == 3 && (aw & 15) == 0 && (af & 3) == 0)
        launch_mode<4>(opt, grid, block, stream, g, in, st, d_density, d_grid, strip, tasks_per_row, (unsigned)n_tasks);
    else if (g.n_p == 2 && g.pol_a == 0 && g.pol_b == 1 && (av & 15) == 0 && (aw & 7) == 0 && (af & 1) == 0)
        launch_mode<2>(opt, grid, block, stream, g, in, st, d_density, d_grid, strip, tasks_per_row, (unsigned)n_tasks);
    else
        launch_mode<0>(-1, grid, block, stream, g, in, st, d_density, d_grid, strip, tasks_per_row, (unsigned)n_tasks);
}

}  // namespace toi
