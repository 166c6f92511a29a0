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
//    average, 14 kernel taps, packed for both axes, square root and exp2 on the MUFU pipe) into
//    an 80-byte shared-memory record each; the groups then consume their 8 records with
//    immediate-offset LDS.  The raw inputs of the next batch are requested before the current one
//    is processed (register prefetch), so HBM latency overlaps a whole batch of arithmetic.
//    Tasks (baseline, block of 4 strips) come from an atomic queue; the grid is persistent.
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
constexpr int kRecQuads = 5;      // record = 5 x 16 B: {zre, zim, key, -} {pu0..3} {pu4..6, -} {pv0..3} {pv4..6, -}
constexpr int kGroupQuads = kBatch * kRecQuads + 2;   // +32 B: groups land on distinct banks
constexpr int kWarpQuads = kGroups * kGroupQuads;
#ifndef KUNROLL
#define KUNROLL 1
#endif
constexpr int kUnroll = KUNROLL;   // records consumed per copy of the accumulate loop body
constexpr int kModBias = 7 << 20; // makes (x + kModBias) % 7 a mathematical mod for |x| < 2^22
constexpr unsigned kNoKey = 0x80008000u;   // (iv, iu) = (-32768, -32768): never an on-grid cell

// centre cell packed into one word: one compare per sample decides "same footprint as before"
__device__ __forceinline__ unsigned cell_key(int iu, int iv) { return ((unsigned)iv << 16) | ((unsigned)iu & 0xffffu); }
__device__ __forceinline__ int key_u(unsigned k) { return (int)(k << 16) >> 16; }
__device__ __forceinline__ int key_v(unsigned k) { return (int)k >> 16; }

__device__ __forceinline__ void red_cell(float2 *cell, u64 v)
{
    const float2 f = unpack2(v);
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(cell), "f"(f.x), "f"(f.y) : "memory");
}

// Flush one window column (7 rows, row stride rs bytes, first row at p) and zero it.  One asm
// block: the accumulators stay in their register pairs and the address walks by one 64-bit add.
__device__ __forceinline__ void flush_col(u64 (&a)[kW], const char *p, long long rs)
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
        "mov.b64 {x, y}, %6;\n\tred.global.add.v2.f32 [p], {x, y};\n\t"
        "mov.b64 %0, 0;\n\tmov.b64 %1, 0;\n\tmov.b64 %2, 0;\n\tmov.b64 %3, 0;\n\t"
        "mov.b64 %4, 0;\n\tmov.b64 %5, 0;\n\tmov.b64 %6, 0;\n\t}"
        : "+l"(a[0]), "+l"(a[1]), "+l"(a[2]), "+l"(a[3]), "+l"(a[4]), "+l"(a[5]), "+l"(a[6])
        : "l"(p), "l"(rs)
        : "memory");
}

// The window moves by (du, dv), each in {-1, 0, 1}: retire one column (the lane that holds it
// flushes 7 cells and takes over the entering column) and/or one row (every lane flushes one cell,
// the row accumulators shift by one register).  p = &grid[cv-3][my column], rs = row stride in
// bytes, mydu = which tap column this lane holds.  One predicated asm block, so that ptxas keeps
// the seven accumulators in place instead of copying them around the branches.
__device__ __forceinline__ void slide_window(u64 (&a)[kW], const char *&p, int &mydu, int du, int dv, long long rs)
{
    asm volatile(
        "{\n\t.reg .pred pc, pu, pd;\n\t.reg .u64 q;\n\t.reg .f32 x, y;\n\t.reg .s32 t;\n\t"
        "setp.gt.s32 pu, %9, 0;\n\t"
        "selp.s32 t, 0, 6, pu;\n\t"
        "setp.ne.s32 pc, %9, 0;\n\t"
        "setp.eq.and.s32 pc, %8, t, pc;\n\t"
        "@!pc bra NOCOL;\n\t"
        "mov.u64 q, %7;\n\t"
        "mov.b64 {x, y}, %0;\n\tred.global.add.v2.f32 [q], {x, y};\n\tadd.s64 q, q, %11;\n\t"
        "mov.b64 {x, y}, %1;\n\tred.global.add.v2.f32 [q], {x, y};\n\tadd.s64 q, q, %11;\n\t"
        "mov.b64 {x, y}, %2;\n\tred.global.add.v2.f32 [q], {x, y};\n\tadd.s64 q, q, %11;\n\t"
        "mov.b64 {x, y}, %3;\n\tred.global.add.v2.f32 [q], {x, y};\n\tadd.s64 q, q, %11;\n\t"
        "mov.b64 {x, y}, %4;\n\tred.global.add.v2.f32 [q], {x, y};\n\tadd.s64 q, q, %11;\n\t"
        "mov.b64 {x, y}, %5;\n\tred.global.add.v2.f32 [q], {x, y};\n\tadd.s64 q, q, %11;\n\t"
        "mov.b64 {x, y}, %6;\n\tred.global.add.v2.f32 [q], {x, y};\n\t"
        "mov.b64 %0, 0;\n\tmov.b64 %1, 0;\n\tmov.b64 %2, 0;\n\tmov.b64 %3, 0;\n\t"
        "mov.b64 %4, 0;\n\tmov.b64 %5, 0;\n\tmov.b64 %6, 0;\n\t"
        "mad.wide.s32 %7, %9, 56, %7;\n\t"
        "mad.lo.s32 %8, %9, 7, %8;\n\t"
        "NOCOL:\n\t"
        "sub.s32 %8, %8, %9;\n\t"
        "setp.gt.s32 pu, %10, 0;\n\t"
        "setp.lt.s32 pd, %10, 0;\n\t"
        "@!pu bra NOUP;\n\t"
        "mov.b64 {x, y}, %0;\n\t"
        "red.global.add.v2.f32 [%7], {x, y};\n\t"
        "mov.b64 %0, %1;\n\tmov.b64 %1, %2;\n\tmov.b64 %2, %3;\n\tmov.b64 %3, %4;\n\t"
        "mov.b64 %4, %5;\n\tmov.b64 %5, %6;\n\tmov.b64 %6, 0;\n\t"
        "add.s64 %7, %7, %11;\n\t"
        "NOUP:\n\t"
        "@!pd bra NODN;\n\t"
        "mad.lo.s64 q, %11, 6, %7;\n\t"
        "mov.b64 {x, y}, %6;\n\t"
        "red.global.add.v2.f32 [q], {x, y};\n\t"
        "mov.b64 %6, %5;\n\tmov.b64 %5, %4;\n\tmov.b64 %4, %3;\n\tmov.b64 %3, %2;\n\t"
        "mov.b64 %2, %1;\n\tmov.b64 %1, %0;\n\tmov.b64 %0, 0;\n\t"
        "sub.s64 %7, %7, %11;\n\t"
        "NODN:\n\t}"
        : "+l"(a[0]), "+l"(a[1]), "+l"(a[2]), "+l"(a[3]), "+l"(a[4]), "+l"(a[5]), "+l"(a[6]),
          "+l"(p), "+r"(mydu)
        : "r"(du), "r"(dv), "l"(rs)
        : "memory");
}

// Raw inputs of one sample as they sit in HBM (requested one batch ahead).
struct Raw {
    float2 a, b;      // the two parallel hands
    float wa, wb;
    unsigned fl;      // bit 0: hand a flagged, bit 1: hand b flagged
    double s;         // s_c = nu_c / c0
};

// MODE 4: n_p = 4, hands (0, 3), 16-B aligned weights and 4-B aligned flags -> 2 LDG.64 + LDG.128 + LDG.32
// MODE 2: n_p = 2, hands (0, 1), 8-B aligned weights, 2-B aligned flags     -> LDG.128 + LDG.64 + LDG.U16
// MODE 0: anything else, scalar loads
template <int MODE>
__device__ __forceinline__ void load_raw(const Geometry &g, const Inputs &in, long long q, int c, Raw &r)
{
    r.s = __ldg(g.s + c);
    if (MODE == 4) {
        const float2 *v = in.vis + 4 * q;
        r.a = __ldg(v);
        r.b = __ldg(v + 3);
        r.wa = r.wb = 1.0f;
        if (in.weights) {
            const float4 w = __ldg(reinterpret_cast<const float4 *>(in.weights) + q);
            r.wa = w.x; r.wb = w.w;
        }
        r.fl = 0u;
        if (in.flags) {
            const unsigned f = __ldg(reinterpret_cast<const unsigned *>(in.flags) + q);
            r.fl = ((f & 0xffu) ? 1u : 0u) | ((f >> 24) ? 2u : 0u);
        }
    } else if (MODE == 2) {
        const float4 v = __ldg(reinterpret_cast<const float4 *>(in.vis) + q);
        r.a = make_float2(v.x, v.y);
        r.b = make_float2(v.z, v.w);
        r.wa = r.wb = 1.0f;
        if (in.weights) {
            const float2 w = __ldg(reinterpret_cast<const float2 *>(in.weights) + q);
            r.wa = w.x; r.wb = w.y;
        }
        r.fl = 0u;
        if (in.flags) {
            const unsigned f = __ldg(reinterpret_cast<const unsigned short *>(in.flags) + q);
            r.fl = ((f & 0xffu) ? 1u : 0u) | ((f >> 8) ? 2u : 0u);
        }
    } else {
        const long long o = q * g.n_p;
        r.a = __ldg(in.vis + o + g.pol_a);
        r.b = __ldg(in.vis + o + g.pol_b);
        r.wa = r.wb = 1.0f;
        if (in.weights) { r.wa = __ldg(in.weights + o + g.pol_a); r.wb = __ldg(in.weights + o + g.pol_b); }
        r.fl = 0u;
        if (in.flags) r.fl = (__ldg(in.flags + o + g.pol_a) ? 1u : 0u) | (__ldg(in.flags + o + g.pol_b) ? 2u : 0u);
        if (g.pol_b == g.pol_a) r.fl |= 2u;     // single hand: b never contributes
    }
}

template <int MODE>
__global__ void __launch_bounds__(kWarps * 32, 3)
k_grid_sliding(Geometry g, Inputs in, SnapState *__restrict__ st, const float *__restrict__ D,
               float2 *__restrict__ grid, int strip_len, int tasks_per_row, unsigned n_tasks)
{
    __shared__ uint4 s_rec[kWarps * kWarpQuads];
    if (st->status != TOI_OK) return;
    const int lane = threadIdx.x & 31;
    uint4 *rec = s_rec + (threadIdx.x >> 5) * kWarpQuads;

    // roles: every lane pre-processes one sample per batch (strip pre_g, channel pre_k of the
    // batch: 8 consecutive samples per strip = 256 contiguous bytes of visibilities); lanes 0..27
    // accumulate (group grp = strip, lane m of the group = one column of the footprint)
    const int pre_g = lane >> 3, pre_k = lane & 7;
    uint4 *my_rec = rec + pre_g * kGroupQuads + pre_k * kRecQuads;
    const bool acc_lane = lane < 7 * kGroups;
    const int grp = acc_lane ? lane / 7 : 0, m = lane - 7 * grp;
    const uint4 *rg = rec + grp * kGroupQuads;
    const int G = g.G;
    float2 *const gc = grid + centre_index(0, 0, G);         // cell (0, 0)
    const long long rs = (long long)G * 8;                   // row stride in bytes
    const float *const Dc = D ? D + centre_index(0, 0, G) : nullptr;

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
        float wpart = 0.0f;

        Raw nxt;
        nxt.a = nxt.b = make_float2(0.0f, 0.0f); nxt.wa = nxt.wb = 0.0f; nxt.fl = 0u; nxt.s = 0.0;
        if (c_lo < c_hi) load_raw<MODE>(g, in, q_row + c_lo, c_lo, nxt);

        for (int b = 0; b < strip_len && c_task + b < g.n_c; b += kBatch) {
            // ---------------- pre-process one sample per lane ----------------
            {
                const int c = c_lo + b;
                const Raw cur = nxt;
                if (c + kBatch < c_hi && b + kBatch < strip_len) load_raw<MODE>(g, in, q_row + c + kBatch, c + kBatch, nxt);
                uint4 q0 = make_uint4(0u, 0u, kNoKey, 0u);
                float pu[kW], pv[kW];
#pragma unroll
                for (int d = 0; d < kW; ++d) pu[d] = pv[d] = 0.0f;
                if (c < c_hi) {
                    int iu, iv;
                    float xu, xv;
                    sample_cell(rho1, rho2, cur.s, g.kappa, iu, iv, xu, xv);
                    if (!cell_on_grid(iu, iv, G)) {
                        ++n_off;
                    } else {
                        const float wa = (weight_ok(cur.wa) && !(cur.fl & 1u)) ? cur.wa : 0.0f;
                        const float wb = (weight_ok(cur.wb) && !(cur.fl & 2u)) ? cur.wb : 0.0f;
                        const float wI = wa + wb;
                        if (!(wI > 0.0f)) {
                            ++n_flag;       // contributes nothing: the record stays "no sample"
                        } else {
                            ++n_grid;
                            float f = 1.0f;
                            if (Dc) {
                                const float dens = __ldg(Dc + ((long long)iv * G + iu));
                                asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(f) : "f"(dens));
                            }
                            // z = w_a Vis_a + w_b Vis_b; a zero-weight hand is skipped (its data may be NaN)
                            float zx = 0.0f, zy = 0.0f;
                            if (wa > 0.0f) { zx = wa * cur.a.x; zy = wa * cur.a.y; }
                            if (wb > 0.0f) { zx = fmaf(wb, cur.b.x, zx); zy = fmaf(wb, cur.b.y, zy); }
                            wpart = fmaf(f, wI, wpart);
                            q0.x = __float_as_uint(zx * f);
                            q0.y = __float_as_uint(zy * f);
                            q0.z = cell_key(iu, iv);
                            kernel_taps2(xu, xv, pu, pv);
                        }
                    }
                }
                my_rec[0] = q0;
                my_rec[1] = make_uint4(__float_as_uint(pu[0]), __float_as_uint(pu[1]), __float_as_uint(pu[2]), __float_as_uint(pu[3]));
                my_rec[2] = make_uint4(__float_as_uint(pu[4]), __float_as_uint(pu[5]), __float_as_uint(pu[6]), 0u);
                my_rec[3] = make_uint4(__float_as_uint(pv[0]), __float_as_uint(pv[1]), __float_as_uint(pv[2]), __float_as_uint(pv[3]));
                my_rec[4] = make_uint4(__float_as_uint(pv[4]), __float_as_uint(pv[5]), __float_as_uint(pv[6]), 0u);
            }
            __syncwarp();
            // ---------------- accumulate: group grp consumes its 8 records ----------------
            if (acc_lane) {
                const char *const rg0 = reinterpret_cast<const char *>(rg);
                const char *rpu = rg0 + 16 + 4 * mydu;              // my tap column in record 0
#pragma unroll kUnroll
                for (int k = 0; k < kBatch; ++k) {
                    const char *const rk = rg0 + k * (kRecQuads * 16);
                    const uint4 q0 = *reinterpret_cast<const uint4 *>(rk);
                    // a "no sample" record (padding / off-grid / flagged) has z = 0 and zero taps: it
                    // falls through the FMAs harmlessly and never moves the window
                    if (__builtin_expect(q0.z != ckey && q0.z != kNoKey, 0)) {
                        const int du = key_u(q0.z) - key_u(ckey), dv = key_v(q0.z) - key_v(ckey);
                        if (ckey != kNoKey && (unsigned)(du + 1) <= 2u && (unsigned)(dv + 1) <= 2u) {
                            slide_window(acc, pcol, mydu, du, dv, rs);
                        } else {                                    // first sample, or a jump
                            if (ckey != kNoKey) flush_col(acc, pcol, rs);
                            const int cu = key_u(q0.z), cv = key_v(q0.z);
                            mydu = (m - cu + kH + kModBias) % kW;   // column (cu-3+mydu) = m (mod 7)
                            pcol = reinterpret_cast<const char *>(gc + ((long long)(cv - kH) * G + (cu - kH + mydu)));
                        }
                        ckey = q0.z;
                        rpu = rg0 + 16 + 4 * mydu;
                    }
                    const float pu = *reinterpret_cast<const float *>(rpu + k * (kRecQuads * 16));
                    const uint4 va = *reinterpret_cast<const uint4 *>(rk + 48), vb = *reinterpret_cast<const uint4 *>(rk + 64);
                    const u64 t = mul2(pack2(__uint_as_float(q0.x), __uint_as_float(q0.y)), pack2(pu, pu));
                    fma2_acc(acc[0], t, pack2(__uint_as_float(va.x), __uint_as_float(va.x)));
                    fma2_acc(acc[1], t, pack2(__uint_as_float(va.y), __uint_as_float(va.y)));
                    fma2_acc(acc[2], t, pack2(__uint_as_float(va.z), __uint_as_float(va.z)));
                    fma2_acc(acc[3], t, pack2(__uint_as_float(va.w), __uint_as_float(va.w)));
                    fma2_acc(acc[4], t, pack2(__uint_as_float(vb.x), __uint_as_float(vb.x)));
                    fma2_acc(acc[5], t, pack2(__uint_as_float(vb.y), __uint_as_float(vb.y)));
                    fma2_acc(acc[6], t, pack2(__uint_as_float(vb.z), __uint_as_float(vb.z)));
                }
            }
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

}  // namespace

void launch_grid_sliding(const Geometry &g, const Inputs &in, SnapState *st, const float *d_density,
                         float2 *d_grid, int n_sms, cudaStream_t stream)
{
    // strip length (channels per group per task): long strips amortise the 49-cell flush at a strip
    // end, short ones balance the persistent grid's tail.  Aim at >= 6 tasks per resident warp,
    // within [32, 256] channels and a multiple of the 8-sample batch.
    const long long warps = 3LL * n_sms * kWarps;
    long long want = ((long long)g.n_b * g.n_c) / (kGroups * 6 * warps);
    want = want / kBatch * kBatch;
    int strip = (int)(want < 32 ? 32 : (want > 256 ? 256 : want));
    const int quarter = ((g.n_c + kGroups - 1) / kGroups + kBatch - 1) / kBatch * kBatch;
    if (strip > quarter) strip = quarter;
    if (const char *e = getenv("TOI_STRIP")) strip = atoi(e);   // tuning override (multiple of 8)
    const int tasks_per_row = (g.n_c + kGroups * strip - 1) / (kGroups * strip);
    const long long n_tasks = (long long)g.n_b * tasks_per_row;
    long long ctas = (n_tasks + kWarps - 1) / kWarps;
    if (ctas > 3LL * n_sms) ctas = 3LL * n_sms;   // persistent: 3 CTAs per SM pull from the queue
    const dim3 grid((unsigned)ctas), block(kWarps * 32);
    const uintptr_t aw = (uintptr_t)in.weights, af = (uintptr_t)in.flags, av = (uintptr_t)in.vis;
    if (g.n_p == 4 && g.pol_a == 0 && g.pol_b == 3 && (aw & 15) == 0 && (af & 3) == 0)
        k_grid_sliding<4><<<grid, block, 0, stream>>>(g, in, st, d_density, d_grid, strip, tasks_per_row, (unsigned)n_tasks);
    else if (g.n_p == 2 && g.pol_a == 0 && g.pol_b == 1 && (av & 15) == 0 && (aw & 7) == 0 && (af & 1) == 0)
        k_grid_sliding<2><<<grid, block, 0, stream>>>(g, in, st, d_density, d_grid, strip, tasks_per_row, (unsigned)n_tasks);
    else
        k_grid_sliding<0><<<grid, block, 0, stream>>>(g, in, st, d_density, d_grid, strip, tasks_per_row, (unsigned)n_tasks);
}

}  // namespace toi
