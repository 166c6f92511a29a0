// k_grid_tma.cu -- step a5, the sliding-window gridder of k_grid_pair8.cu with its raw inputs STAGED
// THROUGH SHARED MEMORY BY TMA (the staging north_star prescribes): one elected lane per warp issues
// three 2-D tensor copies per batch (cp.async.bulk.tensor.2d + mbarrier complete_tx) -- the batch's
// 4 consecutive channels of each of the warp's 8 strips of visibilities [8 x 128 B, 128-byte swizzle],
// weights [8 x 64 B] and flags [8 x 16 B] -- kStages - 1 batches ahead, across task boundaries;
// every lane then reads its own sample with 4 shared-memory loads instead of 5 global loads whose
// register targets had to be carried (and copied) from one batch to the next.
//   grid[iv+dv][iu+du] += f z phi(iu+du-gu) phi(iv+dv-gv),  du, dv = -3..3
// The tensor maps view each input array as [n_b * n_c / strip_len rows][strip_len samples]: the 8
// strips of a task are 8 consecutive rows, a batch is a box of 8 rows x 4 samples.  Needs n_p = 4 with
// hands (0, 3), n_c a multiple of 8 * strip_len, 16-byte aligned arrays; launch_grid_pair8 handles
// everything else.  Pre-processing, records and the consume phase are k_grid_pair8's.
#include <cuda.h>
#include <cudaTypedefs.h>

#include "grid_window.cuh"

namespace toi {
namespace {

constexpr int kWarps = 8;            // warps per CTA
constexpr int kCtasPerSm = 2;
constexpr int kStages = 4;           // batches of raw inputs in flight per warp (3 ahead of the one in use)
constexpr int kVisBytes = 8 * 128, kWBytes = 8 * 64, kFBytes = 8 * 16;
constexpr int kStageBytes = 2048;    // vis 1024 (1024-byte aligned for the 128-byte swizzle) + w 512 + flags 128, padded
constexpr int kWarpStageBytes = kStages * kStageBytes;
constexpr size_t kSmemBytes = (size_t)kWarps * (kWarpStageBytes + kWarpQuads * 16) + kWarps * kStages * 8 + 1024;

__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" : : "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" : : "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@!p bra WAIT_%=;\n\t"
        "}"
        : : "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_2d(unsigned dst, const CUtensorMap *map, int c0, int c1, unsigned bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 : : "r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}

template <int OPT, bool PIPE>
__global__ void __launch_bounds__(kWarps * 32, kCtasPerSm)
k_grid_tma(Geometry g, Inputs in, SnapState *__restrict__ st, const float *__restrict__ D,
           float2 *__restrict__ grid, uint8_t *__restrict__ tiles, int strip_len, int tasks_per_row,
           unsigned n_tasks, const __grid_constant__ CUtensorMap map_vis, const __grid_constant__ CUtensorMap map_w,
           const __grid_constant__ CUtensorMap map_f)
{
    constexpr bool has_w = (OPT & kHasW) != 0, has_f = (OPT & kHasF) != 0, has_d = (OPT & kHasD) != 0;
    constexpr unsigned kTxBytes = kVisBytes + (has_w ? kWBytes : 0) + (has_f ? kFBytes : 0);
    extern __shared__ unsigned char s_dyn[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // shared memory: [stages of all warps, 1024-byte aligned][records of all warps][mbarriers]
    const unsigned s_base = ((unsigned)__cvta_generic_to_shared(s_dyn) + 1023u) & ~1023u;
    const unsigned stage0 = s_base + (unsigned)warp * kWarpStageBytes;
    const unsigned rec_u = s_base + (unsigned)kWarps * kWarpStageBytes + (unsigned)warp * (kWarpQuads * 16);
    const unsigned bar0 = s_base + (unsigned)kWarps * (kWarpStageBytes + kWarpQuads * 16) + (unsigned)warp * (kStages * 8);
    if (lane < kStages) mbar_init(bar0 + 8u * lane, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncwarp();
    if (st->status != TOI_OK) return;

    // every lane pre-processes one sample per batch (strip grp, channel pre_k of the batch) AND
    // accumulates: group grp = lane / 4 = strip, L = lane % 4 = its two column slots L and L + 4
    const int grp = lane >> 2, L = lane & 3;
    const int pre_k = L;
    const unsigned my_rec = rec_u + (unsigned)(group_quad(grp) + pre_k * kRecQuads) * 16u;
    const unsigned rgs = rec_u + (unsigned)group_quad(grp) * 16u;
    // my sample inside a stage: row grp of each tile; the visibilities sit under the 128-byte swizzle
    // (16-byte chunk j of row r is stored at chunk j ^ (r & 7)): hand a = chunk 2L, hand b = chunk 2L + 1, +8 B
    const unsigned off_a = (unsigned)(grp * 128 + (((2 * L) ^ grp) << 4));
    const unsigned off_b = (unsigned)(grp * 128 + (((2 * L + 1) ^ grp) << 4) + 8);
    const unsigned off_w = (unsigned)(kVisBytes + grp * 64 + L * 16);
    const unsigned off_f = (unsigned)(kVisBytes + kWBytes + grp * 16 + L * 4);
    const int G = g.G;
    const float2 *const gc = grid + centre_index(0, 0, G);   // cell (0, 0)
    const long long rs = (long long)G * 8;                   // row stride in bytes
    const float *const Dc = has_d ? D + centre_index(0, 0, G) : nullptr;
    const int n_batches = strip_len / kBatch;                // per task: every strip is full (n_c % (8 strip_len) == 0)

    double wsum = 0.0;
    unsigned n_grid = 0, n_off = 0, n_flag = 0;

    // ---- the fetch cursor (lane 0): runs kStages - 1 batches ahead of the batch being processed,
    // across task boundaries (the next task is claimed while the current one is processed) ----
    unsigned f_task = 0, f_k = 0;            // task and batch the next copy belongs to
    unsigned f_slot = 0;                     // stage it goes to
    unsigned task_ahead = 0;                 // claimed, not yet started
    if (lane == 0) {
        f_task = atomicAdd(&st->task_counter, 1u);
        task_ahead = atomicAdd(&st->task_counter, 1u);
    }
    // first tensor-map row (strip) of a task: rows_per_baseline = 8 * tasks_per_row, so it is 8 * task
    int f_row0 = 0, f_col = 0;               // of the next copy: row0 of its task, channel offset of its batch
    auto fetch_one = [&]() {                 // lane 0 only
        if (f_task >= n_tasks) return;
        const unsigned dst = stage0 + f_slot * kStageBytes, bar = bar0 + 8u * f_slot;
        mbar_expect_tx(bar, kTxBytes);
        tma_load_2d(dst, &map_vis, f_col * 8, f_row0, bar);                             // floats: 8 per sample
        if (has_w) tma_load_2d(dst + kVisBytes, &map_w, f_col * 4, f_row0, bar);
        if (has_f) tma_load_2d(dst + kVisBytes + kWBytes, &map_f, f_col, f_row0, bar);  // one u32 per sample
        if (++f_slot == kStages) f_slot = 0;
        f_col += kBatch;
        if (++f_k == (unsigned)n_batches) { f_k = 0; f_col = 0; f_task = task_ahead; f_row0 = (int)task_ahead * kGroups; }   // on to the claimed task
    };
    unsigned slot = 0, phase = 0;            // stage of the batch being processed
    unsigned task = __shfl_sync(0xffffffffu, f_task, 0);
    if (lane == 0) {
        f_row0 = (int)f_task * kGroups;
        for (int k = 0; k < kStages - 1; ++k) fetch_one();
    }

    while (task < n_tasks) {
        const int j = (int)(task / (unsigned)tasks_per_row);
        const int c_task = (int)(task % (unsigned)tasks_per_row) * (kGroups * strip_len);
        double rho1, rho2;
        rotate_baseline(st->V, in.uvw + 3 * j, rho1, rho2);
        const int c_lo = c_task + grp * strip_len + pre_k;        // my channel in batch 0
        const int c_hi = c_task + (grp + 1) * strip_len;

        // Sparse clear (k_clear.cu): mark the tiles my strip's windows can reach (see k_grid_pair8.cu)
        if (tiles != nullptr) {
            const double s_end = __ldg(g.s + ((L & 1) ? c_hi - 1 : c_task + grp * strip_len));
            const double lim = (double)G;                         // far outside the grid; also absorbs NaN
            const double eu = fmin(fmax(-__dmul_rn(__dmul_rn(rho1, s_end), g.kappa), -lim), lim);
            const double ev = fmin(fmax(__dmul_rn(__dmul_rn(rho2, s_end), g.kappa), -lim), lim);
            const int iu = __double2int_rd(eu + 0.5), iv = __double2int_rd(ev + 0.5);
            const int ju = __shfl_xor_sync(0xffffffffu, iu, 1), jv = __shfl_xor_sync(0xffffffffu, iv, 1);
            if (L == 0) {
                const int h = G >> 1, tpr = tiles_per_row(G);
                const int x0 = max(min(iu, ju) - 4 + h, 0) / kTile, x1 = min(max(iu, ju) + 4 + h, G - 1) / kTile;
                const int y0 = max(min(iv, jv) - 4 + h, 0) / kTile, y1 = min(max(iv, jv) + 4 + h, G - 1) / kTile;
                for (int ty = y0; ty <= y1; ++ty)
                    for (int tx = x0; tx <= x1; ++tx)
                        if (tiles[ty * tpr + tx] == 0) tiles[ty * tpr + tx] = 1;   // L1 hit instead of a store, mostly
            }
        }

        // sliding-window state of my group (ckey uniform across its 4 lanes)
        u64 accA[kR], accB[kR];
#pragma unroll
        for (int d = 0; d < kR; ++d) accA[d] = accB[d] = 0ull;
        unsigned ckey = kNoKey;              // closed window; else the packed base cell (bu, bv)
        unsigned tapA = 0u;                  // window column held by my slot L; slot L + 4 holds tapA ^ 4
        unsigned rpa = rgs + 48, rpb = rgs + 48 + 16;        // shared addresses of my two taps in record 0
        float wpart = 0.0f;

        auto locate = [&](double s_c, Cell &cl) {
            int iu, iv;
            sample_cell(rho1, rho2, s_c, g.kappa, iu, iv, cl.xu, cl.xv);
            cl.key = kNoKey;
            cl.sh = 0u;
            cl.dens = 1.0f;
            if (cell_on_grid(iu, iv, G)) {
                const int bu = (iu - kH) & ~1, bv = (iv - kH) & ~1;
                cl.key = cell_key(bu, bv);
                cl.sh = (unsigned)((iu - kH) & 1) | ((unsigned)((iv - kH) & 1) << 1);
                if (has_d) cl.dens = __ldg(Dc + ((long long)iv * G + iu));
            } else {
                ++n_off;
            }
        };
        // the cell (and, with a density map, its density value: a dependent lookup with L2 latency) of
        // batch b + 1 is computed while batch b is processed; the channel scale runs two batches ahead
        Cell cnxt;
        cnxt.key = kNoKey; cnxt.sh = 0u; cnxt.xu = cnxt.xv = 0.0f; cnxt.dens = 1.0f;
        double s_cur = __ldg(g.s + c_lo), s_ahead = 0.0;
        if (PIPE) {
            locate(s_cur, cnxt);
            if (n_batches > 1) s_ahead = __ldg(g.s + c_lo + kBatch);
        } else if (n_batches > 1) {
            s_ahead = __ldg(g.s + c_lo + kBatch);
        }

        for (int b = 0; b < n_batches; ++b) {
            // keep kStages - 1 batches in flight: the stage freed by the previous batch takes the next copy
            if (lane == 0) fetch_one();
            // ---------------- pre-process one sample per lane ----------------
            {
                Cell cell = cnxt;
                if (PIPE) {
                    if (b + 1 < n_batches) {
                        locate(s_ahead, cnxt);
                        if (b + 2 < n_batches) s_ahead = __ldg(g.s + c_lo + (b + 2) * kBatch);
                    }
                } else {
                    locate(s_cur, cell);
                    s_cur = s_ahead;
                    if (b + 2 < n_batches) s_ahead = __ldg(g.s + c_lo + (b + 2) * kBatch);
                }
                // my raw sample, staged by TMA
                mbar_wait(bar0 + 8u * slot, phase);
                const unsigned sb = stage0 + slot * kStageBytes;
                float2 va, vb;
                float wa_raw = 1.0f, wb_raw = 1.0f;
                unsigned fl = 0u;
                asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(va.x), "=f"(va.y) : "r"(sb + off_a));
                asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(vb.x), "=f"(vb.y) : "r"(sb + off_b));
                if (has_w) {
                    float w1, w2;
                    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(wa_raw), "=f"(w1), "=f"(w2), "=f"(wb_raw) : "r"(sb + off_w));
                }
                if (has_f) asm volatile("ld.shared.u32 %0, [%1];" : "=r"(fl) : "r"(sb + off_f));
                if (++slot == kStages) { slot = 0; phase ^= 1u; }

                unsigned key = kNoKey;
                bool valid = false;
                float wI = 0.0f, zx = 0.0f, zy = 0.0f, pv0 = 0.0f;
                uint4 q1 = make_uint4(0u, 0u, 0u, 0u), q2 = q1, q3 = q1, q4 = q1;
                if (cell.key != kNoKey) {
                    // a flagged sample keeps its own cell as key (z = 0, zero taps): it moves the
                    // window exactly as its unflagged neighbours do and never takes the slow path
                    key = cell.key;
                    const float wa = (weight_ok(wa_raw) && !(fl & 0x000000ffu)) ? wa_raw : 0.0f;
                    const float wb = (weight_ok(wb_raw) && !(fl & 0xff000000u)) ? wb_raw : 0.0f;
                    wI = wa + wb;
                    if (!(wI > 0.0f)) {
                        ++n_flag;
                    } else {
                        ++n_grid;
                        valid = true;
                        // z = w_a Vis_a + w_b Vis_b; a zero-weight hand is skipped (its data may be NaN)
                        if (wa > 0.0f) { zx = wa * va.x; zy = wa * va.y; }
                        if (wb > 0.0f) { zx = fmaf(wb, vb.x, zx); zy = fmaf(wb, vb.y, zy); }
                        float pu[kW], pv[kW];
                        kernel_taps2(cell.xu, cell.xv, pu, pv);
                        // the 7 taps sit at window offset 0 or 1 on each axis; the free end is zero
                        const bool su = (cell.sh & 1u) != 0u, sv = (cell.sh & 2u) != 0u;
                        unsigned wu[kR], wv[kR];
#pragma unroll
                        for (int i = 0; i < kR; ++i) {
                            const float lo_u = i < kW ? pu[i] : 0.0f, hi_u = i > 0 ? pu[i - 1] : 0.0f;
                            const float lo_v = i < kW ? pv[i] : 0.0f, hi_v = i > 0 ? pv[i - 1] : 0.0f;
                            wu[i] = __float_as_uint(su ? hi_u : lo_u);
                            wv[i] = __float_as_uint(sv ? hi_v : lo_v);
                        }
                        pv0 = __uint_as_float(wv[0]);
                        q1 = make_uint4(wv[1], wv[2], wv[3], wv[4]);
                        q2 = make_uint4(wv[5], wv[6], wv[7], 0u);
                        q3 = make_uint4(wu[0], wu[1], wu[2], wu[3]);
                        q4 = make_uint4(wu[4], wu[5], wu[6], wu[7]);
                    }
                }
                float f = 1.0f;
                if (has_d) {
                    // the density of a cell whose samples are all flagged is 0: never invert it
                    const float dens = valid ? cell.dens : 1.0f;
                    asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(f) : "f"(dens));
                }
                wpart = fmaf(f, wI, wpart);
                asm volatile("st.shared.v4.b32 [%0+16], {%1, %2, %3, %4};" : : "r"(my_rec), "r"(q1.x), "r"(q1.y), "r"(q1.z), "r"(q1.w) : "memory");
                asm volatile("st.shared.v4.b32 [%0+32], {%1, %2, %3, %4};" : : "r"(my_rec), "r"(q2.x), "r"(q2.y), "r"(q2.z), "r"(q2.w) : "memory");
                asm volatile("st.shared.v4.b32 [%0+48], {%1, %2, %3, %4};" : : "r"(my_rec), "r"(q3.x), "r"(q3.y), "r"(q3.z), "r"(q3.w) : "memory");
                asm volatile("st.shared.v4.b32 [%0+64], {%1, %2, %3, %4};" : : "r"(my_rec), "r"(q4.x), "r"(q4.y), "r"(q4.z), "r"(q4.w) : "memory");
                asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" : : "r"(my_rec), "r"(__float_as_uint(zx * f)), "r"(__float_as_uint(zy * f)), "r"(key), "r"(__float_as_uint(pv0)) : "memory");
            }
            __syncwarp();
            // ---------------- accumulate: every group consumes its 4 records ----------------
            consume_batch(accA, accB, tapA, ckey, rpa, rpb, rgs, gc, (unsigned)rs, G, L);
            __syncwarp();
        }
        // strip done: flush what is left of the window
        if (ckey != kNoKey) flush_sets(accA, accB, tapA, ckey, gc, rs, G);
        wsum += (double)wpart;
        // the task claimed while this one ran is next; claim another
        task = __shfl_sync(0xffffffffu, task_ahead, 0);
        if (lane == 0 && task < n_tasks) {
            const unsigned claimed = atomicAdd(&st->task_counter, 1u);
            // the fetch cursor (at most kStages - 1 batches ahead: never more than one task) may already
            // be inside `task`; it moves on to the newly claimed one from there
            task_ahead = claimed;
        }
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

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
PFN_cuTensorMapEncodeTiled_v12000 encode_fn()
{
    static PFN_cuTensorMapEncodeTiled_v12000 fn = []() -> PFN_cuTensorMapEncodeTiled_v12000 {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess)
            return nullptr;
        return (PFN_cuTensorMapEncodeTiled_v12000)p;
    }();
    return fn;
}

// [rows][row_elems] of `elem_bytes`-byte elements, box = 8 rows x box_elems
bool make_map(CUtensorMap *m, CUtensorMapDataType dt, int elem_bytes, const void *base, unsigned long long rows,
              unsigned long long row_elems, unsigned box_elems, CUtensorMapSwizzle sw)
{
    const cuuint64_t dims[2] = {row_elems, rows};
    const cuuint64_t strides[1] = {row_elems * (cuuint64_t)elem_bytes};
    const cuuint32_t box[2] = {box_elems, 8u};
    const cuuint32_t estr[2] = {1u, 1u};
    return encode_fn()(m, dt, 2, const_cast<void *>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, sw,
                       CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

// Returns false (and launches nothing) when the shape or the alignment does not fit the TMA path.
bool launch_grid_tma(const Geometry &g, const Inputs &in, SnapState *st, const float *d_density,
                     float2 *d_grid, uint8_t *tiles, int n_sms, cudaStream_t stream)
{
    if (g.n_p != 4 || g.pol_a != 0 || g.pol_b != 3 || !encode_fn()) return false;
    const uintptr_t aw = (uintptr_t)in.weights, af = (uintptr_t)in.flags, av = (uintptr_t)in.vis;
    if ((av & 15) || (aw & 15) || (af & 15)) return false;
    const long long warps = (long long)kCtasPerSm * n_sms * kWarps;
    const long long want = ((long long)g.n_b * g.n_c) / (kGroups * 6 * warps);
    const int strip = pick_strip(g.n_c, kGroups, kBatch, want, 16, 128);
    if (g.n_c % (kGroups * strip) != 0) return false;
    const int tasks_per_row = g.n_c / (kGroups * strip);
    const long long n_tasks = (long long)g.n_b * tasks_per_row;
    if (n_tasks > 0x7fffffffLL) return false;
    const unsigned long long rows = (unsigned long long)g.n_b * (g.n_c / strip);
    CUtensorMap mv, mw, mf;
    if (!make_map(&mv, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, in.vis, rows, (unsigned long long)strip * 8, kBatch * 8, CU_TENSOR_MAP_SWIZZLE_128B))
        return false;
    mw = mv; mf = mv;
    if (in.weights && !make_map(&mw, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, in.weights, rows, (unsigned long long)strip * 4, kBatch * 4, CU_TENSOR_MAP_SWIZZLE_NONE))
        return false;
    if (in.flags && !make_map(&mf, CU_TENSOR_MAP_DATA_TYPE_UINT32, 4, in.flags, rows, (unsigned long long)strip, kBatch, CU_TENSOR_MAP_SWIZZLE_NONE))
        return false;
    long long ctas = (n_tasks + kWarps - 1) / kWarps;
    if (ctas > (long long)kCtasPerSm * n_sms) ctas = (long long)kCtasPerSm * n_sms;   // persistent CTAs pull from the queue
    const dim3 grid((unsigned)ctas), block(kWarps * 32);
    const int opt = (in.weights ? kHasW : 0) | (in.flags ? kHasF : 0) | (d_density ? kHasD : 0);
#define TOI_LAUNCH(O, P)                                                                                              \
    do {                                                                                                              \
        static const cudaError_t once = cudaFuncSetAttribute(k_grid_tma<O, P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes); \
        (void)once;                                                                                                   \
        k_grid_tma<O, P><<<grid, block, kSmemBytes, stream>>>(g, in, st, d_density, d_grid, tiles, strip, tasks_per_row, (unsigned)n_tasks, mv, mw, mf); \
    } while (0)
    switch (opt) {
    case kHasW | kHasF | kHasD: TOI_LAUNCH(kHasW | kHasF | kHasD, true); break;
    case kHasW | kHasF: TOI_LAUNCH(kHasW | kHasF, false); break;
    case kHasW | kHasD: TOI_LAUNCH(kHasW | kHasD, true); break;
    case kHasF | kHasD: TOI_LAUNCH(kHasF | kHasD, true); break;
    case kHasW: TOI_LAUNCH(kHasW, false); break;
    case kHasF: TOI_LAUNCH(kHasF, false); break;
    case kHasD: TOI_LAUNCH(kHasD, true); break;
    default: TOI_LAUNCH(0, false); break;
    }
#undef TOI_LAUNCH
    return true;
}

}  // namespace toi
