// probe_kernels.cuh — kernels of the LASER confidence probe (sm_100a) and what they share with
// flex_kernel.cuh (laser_probe_flex_kernel: the same path with the vocabulary on the MMA M axis).
//
//  laser_probe_fused_kernel   a1 + a2 of include/laser_probe.h: LM-head projection on tcgen05 tensor
//                             cores with the online-softmax statistics (max, lowest-index argmax,
//                             sum-exp) taken straight out of TMEM.  Logits never reach HBM.  Its TAIL
//                             (after a device-wide arrival count) runs the merge of the per-split
//                             statistics, a3 per-request aggregate, a4 threshold (Eq. 5 + clamp) and a5
//                             exit mask on the first min(grid, R) CTAs: one launch per probe call.
//  laser_probe_finalize_kernel  the same merge + a3-a5 as a kernel of its own: laser_probe_combine
//                             (gathered shard statistics), degenerate batches, and the two-kernel
//                             form of a call (LASER_TAIL_SEPARATE).
//
// Orientation: tokens on the MMA M axis (= TMEM lanes), vocabulary on the N axis (= TMEM columns).
// With tcgen05.ld 32x32b every epilogue thread owns one token row and walks its vocabulary columns
// in registers: no cross-lane traffic in the vocabulary loop.
//
// Work decomposition: the vocabulary is cut into tiles of tile_n rows which are dealt round-robin to
// `splits` splits (split sp owns tiles sp, sp + splits, ...: at any moment the CTAs stream one
// contiguous window of W, which HBM serves ~3 % faster than 148 distant ranges); a work item is
// (token tile of 128 rows, split).  Items are ordered token-tile fastest so that CTAs running side
// by side stream the same W rows (one HBM read, L2 hits for the rest).  The grid is persistent
// (<= one CTA per SM); CTA b takes items b, b + grid, ...
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <math_constants.h>

#include <cstdint>
#include <cstdio>

#include "ptx.cuh"

namespace laser {

constexpr int kTileM = 128;       // token rows per MMA (TMEM lanes)
constexpr int kBlockK = 64;       // bf16 elements per k-block = one 128-byte swizzle row
constexpr int kUmmaK = 16;        // K of one tcgen05.mma kind::f16
constexpr int kMaxTileN = 256;    // vocabulary rows per tile (UMMA N <= 256)
constexpr int kMaxStages = 8;
constexpr int kABytes = kTileM * kBlockK * 2;  // 16 KiB of hidden per stage
constexpr int kTmemCols = 512;    // two 256-column accumulators (double buffered)
constexpr int kFusedThreads = 192;  // warp 0 TMA, warp 1 MMA + TMEM alloc, warps 2-5 epilogue
constexpr int kEpilogueThreads = 128;
constexpr int kTailThread0 = 64;    // first epilogue thread: runs the arrival protocol of the tail
constexpr int kMaxFinalizers = 32;  // CTAs of one call that may wait for the arrival count (fused tail)
constexpr int kTailCache = 512;     // requests whose offsets / loads a CTA keeps in shared memory for its tail
constexpr float kLog2e = 1.4426950408889634f;

// How the vocabulary tiles are dealt to the execution units (CTAs, or CTA pairs) for `m_items` token
// items: deal the `total_tiles` tiles of tile_n rows to `splits` splits of at most `T` tiles each such
// that m_items * splits fills the units in whole rounds with the least work on the busiest unit.
// Shared by the host planner and both kernels: when a batch carries padding rows (req_offsets[R] <
// N) the kernels re-plan on the device for the token items that actually hold rows.
// Records of the workspace are packed: (row n, split sp) lives at ws[n * splits + sp] with the split
// count of the plan that actually runs (so the workspace holds max over item counts m of
// m * rows_per_item * plan_splits(m).splits records, not the largest split count times every row).
struct SplitPlan {
    int T, splits;
};
__host__ __device__ inline SplitPlan plan_splits(int total_tiles, int m_items, int units) {
    int a = units, b = m_items;
    while (b) { const int t = a % b; a = b; b = t; }
    const int s_unit = units / a;   // smallest split count that fills whole rounds
    SplitPlan best{total_tiles, 1};
    long best_cost = -1;
    for (int k = 1; k <= 4; ++k) {
        const int s_try = s_unit * k;
        const int T = (total_tiles + s_try - 1) / s_try;
        const int S = (total_tiles + T - 1) / T;
        const long rounds = (static_cast<long>(m_items) * S + units - 1) / units;
        const long cost = rounds * (T * 8 + 1);   // a small charge per round for the item switch
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; best.T = T; best.splits = S; }
    }
    return best;
}

// ---------------------------------------------------------------------------------- call plans
// Mixed schedule (kernel_mode AUTO above 1024 rows, MIXED above 256): the token rows are cut into 128-row tiles; an even
// count runs as 256-row items on CTA pairs (cta_group::2); of an odd count the LAST 128-row tile runs
// on single CTAs (cta_group::1) instead of being padded to a pair item.  cta_group is a property of a
// kernel, so a call is two launches - the single-CTA ("tail-tile") kernel first, the pair kernel
// behind it with programmatic dependent launch - whose CTAs look at req_offsets[R] on the device,
// split the SMs between the two parts in proportion to their work, and exit at once where they have
// nothing to do; both walk W in the same tile order, so the second reader of a W tile finds it in L2.
struct MixedPlan {
    int k_pair, j_single;  // 256-row pair items; 128-row tiles behind them for the single-CTA kernel
    int u_pair, u_tail;    // CTA pairs / single CTAs that take part
    int S_pair, S_tail;    // vocabulary splits per item of either part
};
// The host plans every count m128 of 128-row tiles that may hold rows (laser_probe.cu, fill_mixed_table)
// and hands the kernels one packed word per count: looking the plan up on the device costs nothing.
//   bits [0,2)   schedule: 0 pair items only (an odd count pads half an item), 1 pair items + one
//                single-CTA tile, 2 single-CTA tiles only
//   bits [2,10)  u_tail   bits [10,21)  S_pair   bits [21,32)  S_tail
constexpr int kMixedTabMax = 256;     // counts beyond the table: pair items only, planned on the device
__host__ __device__ inline uint32_t mixed_pack(int sched, int u_tail, int S_pair, int S_tail) {
    return static_cast<uint32_t>(sched) | (static_cast<uint32_t>(u_tail) << 2) |
           (static_cast<uint32_t>(S_pair) << 10) | (static_cast<uint32_t>(S_tail) << 21);
}
__host__ __device__ inline MixedPlan mixed_unpack(uint32_t e, int m128, int sms) {
    MixedPlan mp;
    const int sched = static_cast<int>(e & 3u);
    mp.u_tail = static_cast<int>((e >> 2) & 0xFFu);
    mp.S_pair = static_cast<int>((e >> 10) & 0x7FFu);
    mp.S_tail = static_cast<int>((e >> 21) & 0x7FFu);
    mp.k_pair = sched == 0 ? (m128 + 1) / 2 : (sched == 1 ? m128 / 2 : 0);
    mp.j_single = sched == 0 ? 0 : (sched == 1 ? 1 : m128);
    mp.u_pair = mp.k_pair > 0 ? (sms - mp.u_tail) / 2 : 0;
    return mp;
}

// Flex kernel (flex_kernel.cuh; vocabulary on the MMA M axis, tokens on N): the valid rows are cut into
// C chunks of n_tok rows (a multiple of 16, <= 256 = UMMA N) and every chunk's vocabulary tiles (256 rows
// per CTA pair) into S splits.  The host plans every count of 16-row groups that may hold rows and hands
// the kernel one packed word per count (PlanDesc.mixed_tab, kind 3):
//   bits [0,5) C   bits [5,10) n_tok / 16   bits [10,22) S
constexpr int kFlexVocabTile = 256;   // vocabulary rows per tile and CTA pair (UMMA M of cta_group::2)
constexpr int kFlexMaxTok = 256;      // token rows per chunk
constexpr int kFlexMaxRows = 16 * 256;   // largest batch the table covers
struct FlexPlan {
    int C, n_tok, S;
};
__host__ __device__ inline uint32_t flex_pack(int C, int n_tok, int S) {
    return static_cast<uint32_t>(C) | (static_cast<uint32_t>(n_tok >> 4) << 5) | (static_cast<uint32_t>(S) << 10);
}
__host__ __device__ inline FlexPlan flex_unpack(uint32_t e) {
    return FlexPlan{static_cast<int>(e & 31u), static_cast<int>((e >> 5) & 31u) << 4, static_cast<int>((e >> 10) & 0xFFFu)};
}

// What fixes a call's decomposition; shared by the fused kernel(s) and the merge.
struct PlanDesc {
    int32_t kind;                      // 0 static, 1 re-plan of one variant, 2 mixed (pair + single-CTA tail tile), 3 flex
    int32_t n_alloc, R;
    const int32_t* req_offsets;
    int32_t m_tiles, rows_per_item, splits;    // kind 0 / 1: the host plan of the variant
    int32_t total_tiles, units;                // kind 1: vocabulary tiles of the variant, its execution units
    int32_t tiles_pair, sms;                   // kind 2: vocabulary tiles of the pair kernel, SMs
    uint32_t mixed_tab[kMixedTabMax];          // kind 2: the plan for every count of 128-row tiles (mixed_pack)
                                               // kind 3: for every count of 16-row groups, entry [count - 1] (flex_pack)
};
// Where a call's records are: rows [0, rows_a) have S_a records each from record 0 on; rows >= rows_a
// have S_b records each from record rows_a * S_a on.
struct RecLayout {
    int rows_a, S_a, S_b;
};
// The decomposition that actually runs, decided on the device from req_offsets[R] (kind 1, 2).
struct RunPlan {
    MixedPlan mp;          // kind 2
    int m_items, S;        // kind 0 / 1; kind 3: token chunks C, vocabulary splits S
    int n_tok;             // kind 3: token rows per chunk
    RecLayout lay;
};
__device__ __forceinline__ RunPlan resolve_plan(const PlanDesc& d) {
    RunPlan rp{};
    rp.m_items = d.m_tiles; rp.S = d.splits;
    if (d.kind != 0) {   // uniform across the grid: every thread reads the same word
        const int n_valid = d.R > 0 ? min(max(__ldg(d.req_offsets + d.R), 0), d.n_alloc) : 0;
        if (d.kind == 3) {
            const int g16 = (n_valid + 15) >> 4;
            const FlexPlan fp = g16 > 0 ? flex_unpack(d.mixed_tab[min(g16, kMixedTabMax) - 1]) : FlexPlan{0, 16, 1};
            rp.m_items = fp.C; rp.S = fp.S; rp.n_tok = fp.n_tok;
            // both CTAs of a pair leave a record per (row, split): 2 S records per row
            rp.lay = RecLayout{0x7fffffff, 2 * fp.S, 2 * fp.S};
            return rp;
        }
        if (d.kind == 1) {
            const int m = (n_valid + d.rows_per_item - 1) / d.rows_per_item;
            if (m < d.m_tiles) {
                rp.m_items = m;
                rp.S = m > 0 ? plan_splits(d.total_tiles, m, d.units).splits : 1;
            }
        } else {
            const int m128 = (n_valid + kTileM - 1) / kTileM;
            if (m128 < kMixedTabMax) {
                rp.mp = mixed_unpack(d.mixed_tab[m128], m128, d.sms);
            } else {    // very large batches: an odd last tile is noise, pad it
                const int up = d.sms / 2 > 0 ? d.sms / 2 : 1;
                rp.mp = MixedPlan{(m128 + 1) / 2, 0, up, 0, plan_splits(d.tiles_pair, (m128 + 1) / 2, up).splits, 1};
            }
        }
    }
    if (d.kind == 2) rp.lay = RecLayout{2 * kTileM * rp.mp.k_pair, rp.mp.S_pair, rp.mp.S_tail};
    else rp.lay = RecLayout{0x7fffffff, rp.S, rp.S};
    return rp;
}
__device__ __forceinline__ const float4* row_records(const float4* ws, const RecLayout& L, int n, int& nsplit) {
    if (n < L.rows_a) { nsplit = L.S_a; return ws + static_cast<int64_t>(n) * L.S_a; }
    nsplit = L.S_b;
    return ws + static_cast<int64_t>(L.rows_a) * L.S_a + static_cast<int64_t>(n - L.rows_a) * L.S_b;
}

struct FusedParams {
    int32_t n_alloc, d, V;
    int32_t tile_n, k_blocks, stages;
    int32_t total_tiles;   // vocabulary tiles of tile_n rows (this kernel's variant)
    uint32_t tx_bytes;     // bytes TMA delivers per stage and CTA (hidden box + W box)
    uint32_t stage_bytes;  // shared-memory stride of a stage: kABytes + (W rows per CTA) * 128
    uint64_t w_policy;     // L2 eviction policy for the W stream
    float4* ws;            // packed records {max, sum exp(logit - max), argmax bits, token logit}, see RecLayout
    // LASER_PROB_TOKEN: token_ids[n] - v_offset is the column of W whose logit is kept for row n
    // (nullptr: no token logit is tracked; v_offset = global vocabulary index of W's row 0).
    const int32_t* token_ids;
    int32_t v_offset;
    PlanDesc pd;           // the call's decomposition (padding-aware on the device when pd.kind != 0)
    // 0: the call's only fused kernel.  Mixed schedule: 2 = the single-CTA tail-tile kernel (launched
    // first; it alone orders the call against the kernel ahead: griddepcontrol.wait, THEN
    // launch_dependents), 1 = the pair kernel behind it (never waits before it has counted itself in:
    // kernel 2 may be waiting for its arrivals).
    int32_t role;
    int32_t grid_total;    // one fused kernel: its CTAs, what the tail's arrival count waits for (mixed: TailRole)
    // 1 (strict, default): griddepcontrol.wait before the first read of hidden / req_offsets /
    //    token_ids; W - model weight, never written by the kernel ahead - is requested for the first
    //    `stages` pipeline slots before the wait when the plan is static (pd.kind == 0).
    // 0 (overlap): only the workspace / output stores wait (laser_probe_options.overlap).
    int32_t wait_first;
    // requests whose {offset, threshold} fit in the shared memory the pipeline leaves over: the
    // epilogue warps fill that cache right after the wait, so the tail needs no input loads
    int32_t tail_cache;
    // flex kernel: the decomposition of a batch whose n_alloc rows are all valid (chunks, splits).  The
    // producer requests the W boxes of its first tiles under this guess ahead of the wait; when
    // req_offsets[R] then says otherwise the boxes are dropped (0: nothing is requested early).
    int32_t hint_C, hint_S;
    // W layout (laser_probe_options.w_layout).  0: row-major [V, d].  V (> 0): K-block-major
    // [ceil(d/64)][V][64] (laser_probe_pack_w): the tensor map sees k_blocks * V rows of 64 columns, the box
    // of (k-block kb, W row r) is at row kb * V + r and is ONE contiguous run of bytes in HBM.
    int32_t w_kb_rows;
    // W boxes the producer asks L2 for ahead of the wait, behind the `stages` boxes it requests into shared memory
    int32_t prefetch_slots;
    int32_t early_w;          // 1: W boxes may be requested ahead of griddepcontrol.wait (strict calls whose W is not produced on the stream)
};
__device__ __forceinline__ int w_c0(const FusedParams& p, int kb) { return p.w_kb_rows ? 0 : kb * kBlockK; }
__device__ __forceinline__ int w_c1(const FusedParams& p, int kb, int row) { return row + kb * p.w_kb_rows; }

// ---------------------------------------------------------------------------------- descriptors
// Shared-memory matrix descriptor, K-major operand, 128-byte swizzle: rows of 128 B, 8-row groups
// 1024 B apart (SBO), LBO unused for swizzled K-major, descriptor version 1 (Blackwell).
__device__ __forceinline__ uint64_t make_smem_desc_sw128(uint32_t smem_addr) {
    uint64_t desc = 0;
    desc |= static_cast<uint64_t>((smem_addr & 0x3FFFFu) >> 4);   // start address  [0,14)
    desc |= static_cast<uint64_t>(1024u >> 4) << 32;              // SBO            [32,46)
    desc |= static_cast<uint64_t>(1) << 46;                       // version        [46,48)
    desc |= static_cast<uint64_t>(2) << 61;                       // SWIZZLE_128B   [61,64)
    return desc;
}
// Instruction descriptor for kind::f16: D fp32, A/B bf16, both K-major, M = m (128, or 256 for a
// cta_group::2 pair), N = tile_n.
__device__ __forceinline__ uint32_t make_idesc_bf16(uint32_t n, uint32_t m) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((n >> 3) << 17) | ((m >> 4) << 24);
}

// ---------------------------------------------------------------------------------- epilogue math
// Fold NC consecutive vocabulary columns (starting at vocabulary index vbase) of one token row into
// the running statistics (m, a, s):  m = max, a = lowest index attaining it, s = sum 2^{(x-m)log2e}.
// Columns are visited in ascending vocabulary order and the update is strict (>), so ties keep the
// lowest index.  Columns v >= V (TMA zero fill past the end of W) are masked out.
// tok is the row's token column (LASER_PROB_TOKEN; negative = none): its logit is copied to lt when
// this chunk holds it (once per row and vocabulary sweep).
template <int NC>
__device__ __forceinline__ void fold_columns(const uint32_t (&r)[NC], int vbase, int V, float& m,
                                             int& a, float& s, int tok, float& lt) {
    float x[NC];
#pragma unroll
    for (int j = 0; j < NC; ++j) x[j] = __uint_as_float(r[j]);
    if (vbase + NC > V) {
#pragma unroll
        for (int j = 0; j < NC; ++j)
            if (vbase + j >= V) x[j] = -CUDART_INF_F;
    }
    const unsigned dt = static_cast<unsigned>(tok - vbase);
    if (dt < static_cast<unsigned>(NC)) {
#pragma unroll
        for (int j = 0; j < NC; ++j)
            if (static_cast<unsigned>(j) == dt) lt = x[j];
    }
    float c0 = x[0], c1 = x[1], c2 = x[2], c3 = x[3];
#pragma unroll
    for (int j = 4; j < NC; j += 4) {
        c0 = fmaxf(c0, x[j]);
        c1 = fmaxf(c1, x[j + 1]);
        c2 = fmaxf(c2, x[j + 2]);
        c3 = fmaxf(c3, x[j + 3]);
    }
    const float cm = fmaxf(fmaxf(c0, c1), fmaxf(c2, c3));
    if (cm > m) {
        int idx = 0;
#pragma unroll
        for (int j = NC - 1; j >= 0; --j)
            if (x[j] == cm) idx = j;
        a = vbase + idx;
        s *= ptx::ex2_approx((m - cm) * kLog2e);  // m = -inf on the first chunk: s = 0 stays 0
        m = cm;
    }
    const float ms = m * kLog2e;
    float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
#pragma unroll
    for (int j = 0; j < NC; j += 4) {
        s0 += ptx::ex2_approx(fmaf(x[j], kLog2e, -ms));
        s1 += ptx::ex2_approx(fmaf(x[j + 1], kLog2e, -ms));
        s2 += ptx::ex2_approx(fmaf(x[j + 2], kLog2e, -ms));
        s3 += ptx::ex2_approx(fmaf(x[j + 3], kLog2e, -ms));
    }
    s += (s0 + s1) + (s2 + s3);
}

// ---------------------------------------------------------------------------------- finalize
struct TauParamsDev {
    float lambda_base, beta, gamma, l_target, lambda_min, lambda_max;
};

// a4: Eq. 5 then the clamp.  Shared by the kernels and laser_tau_from_load.
__host__ __device__ __forceinline__ float tau_eval(float load, const TauParamsDev& t) {
    float lam = t.lambda_base - t.beta * tanhf(t.gamma * (load - t.l_target) / t.l_target);
    lam = fmaxf(lam, t.lambda_min);
    lam = fminf(lam, t.lambda_max);
    return lam;
}

// One 16-byte record of online-softmax statistics: what the fused kernel leaves per (row, split) in
// the workspace, what laser_probe_partial leaves per row of a vocabulary shard, and what
// laser_probe_combine merges.  Same layout as laser_row_stats in include/laser_probe.h.
//   x = max logit, y = sum exp(logit - max), z = argmax (int bits), w = logit of the row's token
struct FinalizeParams {
    int32_t n_alloc, R, agg_mode;
    PlanDesc pd;      // where the fused kernel(s) left the records (packed workspace: row_stride == 0)
    // gathered shard statistics [G, N] (laser_probe_combine): record (n, g) at ws[n * row_stride +
    // g * split_stride] with row_stride = 1, split_stride = N, pd.kind = 0, pd.splits = G
    int64_t row_stride, split_stride;
    int32_t prob_mode;            // 0: row maximum 1/S; 1: the row's token exp(l_tok - m)/S
    int32_t a_offset;             // added to every argmax (vocabulary shard offset; reduce path)
    // laser_probe_combine over peer-pushed statistics: wait until flags[g] has reached `epoch` for
    // every g < splits before reading (nullptr: the records are already complete in stream order).
    const uint32_t* wait_flags;
    uint32_t epoch;
    const float4* ws;
    const int32_t* req_offsets;
    const float* load;
    float* out_conf;
    int32_t* out_argmax;
    uint8_t* out_exit;
    float* out_tau;   // nullable
    float* out_pmax;  // nullable
    TauParamsDev tau;
};

constexpr int kFinalizeThreads = 256;
constexpr int kFinalizeWarps = kFinalizeThreads / 32;
constexpr int kMaxTailWarps = 8;
constexpr int kMergeBatch = 5;  // partials a lane loads before it starts merging (148 splits: one batch)

// Merge the nsplit records of each of NR rows across a warp (lanes stride over the records; the loads
// of all NR rows are issued before the first merge so that they overlap - one L2 round trip instead
// of NR; then shuffles).  rec[i] == nullptr skips row i.  Every lane returns the merged statistics.
// The records may have been written by other CTAs of the running grid (tail of the fused kernel):
// they are read through L2 (ld.global.cg), never through this SM's L1.
template <int NR>
__device__ __forceinline__ void merge_rows(const float4* const (&rec)[NR], int64_t split_stride,
                                           const int (&ns)[NR], int lane, float (&m)[NR], int (&a)[NR],
                                           float (&s)[NR], float (&lt)[NR]) {
    int nsplit = 0;
#pragma unroll
    for (int i = 0; i < NR; ++i) nsplit = max(nsplit, rec[i] != nullptr ? ns[i] : 0);
    const float4 neutral = make_float4(-CUDART_INF_F, 0.f, __int_as_float(0x7fffffff), -CUDART_INF_F);
    // 2^{(x - M) log2e} with the convention that equal operands (also -inf, -inf) give exactly 1
    auto scale = [](float x, float M) { return (x == M) ? 1.f : ptx::ex2_approx((x - M) * kLog2e); };
#pragma unroll
    for (int i = 0; i < NR; ++i) { m[i] = -CUDART_INF_F; s[i] = 0.f; lt[i] = -CUDART_INF_F; a[i] = 0x7fffffff; }
    // ---- this lane's records: maximum first, then ONE rescale per record (independent ex2, no
    // dependent chain of pairwise merges); on equal maxima the smaller vocabulary index wins
    for (int sp0 = lane; sp0 < nsplit; sp0 += 32 * kMergeBatch) {
        float4 v[NR][kMergeBatch];
#pragma unroll
        for (int i = 0; i < NR; ++i)
#pragma unroll
            for (int j = 0; j < kMergeBatch; ++j) {
                const int sp = sp0 + 32 * j;
                v[i][j] = (rec[i] != nullptr && sp < ns[i]) ? __ldcg(rec[i] + sp * split_stride) : neutral;
            }
#pragma unroll
        for (int i = 0; i < NR; ++i) {
            float M = m[i];
#pragma unroll
            for (int j = 0; j < kMergeBatch; ++j) M = fmaxf(M, v[i][j].x);
            float sum = s[i] * scale(m[i], M);
            int am = (m[i] == M) ? a[i] : 0x7fffffff;
#pragma unroll
            for (int j = 0; j < kMergeBatch; ++j) {
                sum += v[i][j].y * scale(v[i][j].x, M);
                am = (v[i][j].x == M) ? min(am, __float_as_int(v[i][j].z)) : am;
                lt[i] = fmaxf(lt[i], v[i][j].w);
            }
            m[i] = M; s[i] = sum; a[i] = am;
        }
    }
    // ---- across the warp: max, then one rescale per lane, then plain sum / min / max reductions
#pragma unroll
    for (int i = 0; i < NR; ++i) {
        float M = m[i];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, off));
        s[i] *= scale(m[i], M);
        a[i] = (m[i] == M) ? a[i] : 0x7fffffff;
        m[i] = M;
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
        for (int i = 0; i < NR; ++i) {
            s[i] += __shfl_xor_sync(0xffffffffu, s[i], off);
            a[i] = min(a[i], __shfl_xor_sync(0xffffffffu, a[i], off));
            lt[i] = fmaxf(lt[i], __shfl_xor_sync(0xffffffffu, lt[i], off));
        }
    }
}
__device__ __forceinline__ void merge_row(const float4* rec, int64_t split_stride, int nsplit, int lane,
                                          float& m, int& a, float& s, float& lt) {
    const float4* const r1[1] = {rec};
    const int n1[1] = {nsplit};
    float mm[1], ss[1], ll[1];
    int aa[1];
    merge_rows<1>(r1, split_stride, n1, lane, mm, aa, ss, ll);
    m = mm[0]; a = aa[0]; s = ss[0]; lt = ll[0];
}

// Records of row n: packed workspace (layout decided on the device) or gathered shard statistics.
__device__ __forceinline__ const float4* finalize_row(const FinalizeParams& p, const RecLayout& lay, int n,
                                                      int& nsplit) {
    if (p.row_stride != 0) { nsplit = lay.S_a; return p.ws + static_cast<int64_t>(n) * p.row_stride; }
    return row_records(p.ws, lay, n, nsplit);
}

// Spin until every peer's flag has reached `epoch` (peer GPUs store them with system scope after
// their statistics have landed here).  One thread per flag, then a block barrier.
__device__ __forceinline__ void wait_peer_flags(const uint32_t* flags, int G, uint32_t epoch) {
    if (static_cast<int>(threadIdx.x) < G) {
        const long long t0 = clock64();
        while (static_cast<int32_t>(ptx::ld_acquire_sys_u32(flags + threadIdx.x) - epoch) < 0) {
            __nanosleep(64);
            // a peer that never signals (crashed rank, mismatched epoch) must not hang the GPU:
            // after ~5 s the kernel traps and the caller sees a CUDA error instead
            if (clock64() - t0 > 10000000000LL) __trap();
        }
    }
    __syncthreads();
}

// Barrier of a thread group: the whole block (kBarId == 0) or kThreads threads on named barrier kBarId
// (the four epilogue warps in the tail of the fused kernel).
template <int kBarId, int kThreads>
__device__ __forceinline__ void group_sync() {
    if constexpr (kBarId == 0) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"n"(kBarId), "n"(kThreads) : "memory");
}

// Merge + a3 + a4 + a5 of request r by a thread group of nwarps warps (every thread of the group must
// call this, it contains group barriers; tid = index in the group).  A warp takes rows b+w, b+w+nwarps, ...: its
// lanes stride over the records of the row, fold their own, then merge across the warp with shuffles.
// warp_acc: shared scratch of nwarps floats.  [b, e) = the request's rows (every thread), tau = its
// threshold (needed in thread kFinalThread only): the callers read them before they wait for the
// records, so that those loads are off the critical path.
constexpr int kFinalThread = 32;   // lane 0 of the group's warp 1 (thread 0 runs the arrival protocol in the tail)
template <int kBarId, int kThreads>
__device__ __forceinline__ void finalize_request(const FinalizeParams& p, int tid, int r, int b, int e, float tau,
                                                 const RecLayout& lay, float* warp_acc) {
    constexpr int nwarps = kThreads / 32;
    const int warp = tid >> 5, lane = tid & 31;
    // running aggregate of this warp's rows: sum (mean), sum of logs (geomean), min.  Two rows per
    // pass (rows n and n + nwarps): their record loads share one L2 round trip.
    float acc = (p.agg_mode == 2) ? CUDART_INF_F : 0.f;
    bool any_nan = false;
    for (int n0 = b + warp; n0 < e; n0 += 2 * nwarps) {
        const int n1 = n0 + nwarps;
        int ns[2] = {0, 0};
        const float4* const rec[2] = {finalize_row(p, lay, n0, ns[0]),
                                      n1 < e ? finalize_row(p, lay, n1, ns[1]) : nullptr};
        float m[2], s[2], lt[2];
        int a[2];
        merge_rows<2>(rec, p.split_stride, ns, lane, m, a, s, lt);
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const int n = i == 0 ? n0 : n1;
            if (n >= e) break;
            // s >= 1 up to the rounding of ex2.approx; a probability does not exceed 1.  NaN stays NaN.
            float prob;
            if (p.prob_mode == 0) {
                prob = (s[i] == s[i]) ? fminf(1.0f / s[i], 1.0f) : CUDART_NAN_F;
            } else {   // the row's token: exp(l_tok - m) / S; a token outside the vocabulary has l_tok = -inf -> 0
                prob = (s[i] == s[i]) ? fminf(ptx::ex2_approx((lt[i] - m[i]) * kLog2e) / s[i], 1.0f) : CUDART_NAN_F;
            }
            if (lane == 0) {
                p.out_argmax[n] = a[i];
                if (p.out_pmax) p.out_pmax[n] = prob;
            }
            any_nan |= (prob != prob);
            if (p.agg_mode == 0) acc += prob;
            else if (p.agg_mode == 1) acc += logf(prob);
            else acc = fminf(acc, prob);
        }
    }
    if (p.agg_mode == 2 && any_nan) acc = CUDART_NAN_F;
    if (lane == 0) warp_acc[warp] = acc;
    group_sync<kBarId, kThreads>();
    if (tid == kFinalThread) {
        const int len = e - b;
        float conf = 0.f;
        if (len > 0) {
            if (p.agg_mode == 2) {
                conf = warp_acc[0];
                bool nan = conf != conf;
                for (int w = 1; w < nwarps; ++w) {
                    nan |= (warp_acc[w] != warp_acc[w]);
                    conf = fminf(conf, warp_acc[w]);
                }
                if (nan) conf = CUDART_NAN_F;
            } else {
                float t = 0.f;
                for (int w = 0; w < nwarps; ++w) t += warp_acc[w];
                conf = t / static_cast<float>(len);
                if (p.agg_mode == 1) conf = expf(conf);
            }
        }
        p.out_conf[r] = conf;                  // a3
        p.out_exit[r] = (conf > tau) ? 1 : 0;  // a5: strict; NaN > tau is false
        if (p.out_tau) p.out_tau[r] = tau;
    }
    group_sync<kBarId, kThreads>();   // warp_acc may be reused by the caller's next request
}

// Outputs of padding rows (n >= req_offsets[R]): argmax -1, pmax NaN.  Rows are dealt to threads
// `first`, `first + step`, ... of [n_valid, n_alloc).
__device__ __forceinline__ void mark_padding_rows(const FinalizeParams& p, int first, int step) {
    const int n_valid = (p.R > 0) ? min(max(__ldg(p.req_offsets + p.R), 0), p.n_alloc) : 0;
    for (int n = n_valid + first; n < p.n_alloc; n += step) {
        p.out_argmax[n] = -1;
        if (p.out_pmax) p.out_pmax[n] = CUDART_NAN_F;
    }
}

// Standalone form.  Blocks [0, R): one request each.  Blocks [R, R + ceil(n_alloc/256)): mark padding
// rows.  Every global store comes after griddepcontrol.wait (the kernel ahead in the stream may be a
// previous call still writing the same output buffers).
__global__ void __launch_bounds__(kFinalizeThreads)
laser_probe_finalize_kernel(const __grid_constant__ FinalizeParams p) {
    __shared__ float warp_acc[kFinalizeWarps];
    ptx::pdl_launch_dependents();
    if (static_cast<int>(blockIdx.x) >= p.R) {
        ptx::pdl_wait();
        const int nb = gridDim.x - p.R;
        mark_padding_rows(p, (blockIdx.x - p.R) * kFinalizeThreads + threadIdx.x, nb * kFinalizeThreads);
        return;
    }
    // inputs of the probe call, complete before its first kernel started: read ahead of the wait
    const int r = blockIdx.x;
    const int b = __ldg(p.req_offsets + r), e = __ldg(p.req_offsets + r + 1);
    float tau = 0.f;
    if (threadIdx.x == kFinalThread) tau = tau_eval(__ldg(p.load + r), p.tau);   // a4
    ptx::pdl_wait();  // all of the fused kernel's partials are visible after this
    const RunPlan rp = resolve_plan(p.pd);
    if (p.wait_flags != nullptr) wait_peer_flags(p.wait_flags, p.pd.splits, p.epoch);
    finalize_request<0, kFinalizeThreads>(p, threadIdx.x, r, b, e, tau, rp.lay, warp_acc);
}

// ---------------------------------------------------------------------------------- vocab-parallel
// laser_probe_partial: the fused kernel over one vocabulary SHARD; its tail (or, in the two-kernel
// form, laser_probe_reduce_kernel) merges each row's split records into a single record
// {m, S, argmax + v_offset, l_tok} and stores it
//   * to out_stats[n] (local), and
//   * when peers are given, to slot [rank, n] of every GPU's gathered buffer [G, N] through
//     peer-mapped pointers (NVLink stores; 16 bytes per row and peer) - the all-gather of the
//     statistics is done by the producer, no collective call.
// Rows n >= req_offsets[R] (padding) get the neutral record.  When every row has been pushed,
// `epoch` is published in slot [rank] of every GPU's flag array (system-scope release).
constexpr int kMaxPeers = 16;
struct ReduceParams {
    FinalizeParams f;          // ws, strides, replan fields, req_offsets, R, n_alloc, a_offset
    float4* out_stats;         // [n_alloc] or nullptr
    int32_t rank, world;       // world = 0: no peers
    uint32_t epoch;
    float4* peer_stats[kMaxPeers];   // peer_stats[g] = base of GPU g's gathered buffer [world, n_alloc]
    uint32_t* peer_flags[kMaxPeers]; // peer_flags[g] = GPU g's flag array [world]
};

// One warp: merged record of row n -> out_stats / peers.
__device__ __forceinline__ void reduce_row(const ReduceParams& q, int n, int n_valid, const RecLayout& lay,
                                           int lane) {
    const FinalizeParams& p = q.f;
    float m = -CUDART_INF_F, s = 0.f, lt = -CUDART_INF_F;
    int a = 0x7fffffff;
    if (n < n_valid) {
        int nsplit = 0;
        const float4* rec = finalize_row(p, lay, n, nsplit);
        merge_row(rec, p.split_stride, nsplit, lane, m, a, s, lt);
        a += p.a_offset;
    }
    const float4 rec = make_float4(m, s, __int_as_float(a), lt);
    if (lane == 0 && q.out_stats) q.out_stats[n] = rec;
    if (lane < q.world) q.peer_stats[lane][static_cast<int64_t>(q.rank) * p.n_alloc + n] = rec;
}

__device__ __forceinline__ void publish_epoch(const ReduceParams& q, int lane) {
    if (lane < q.world) {
        __threadfence_system();
        ptx::st_release_sys_u32(q.peer_flags[lane] + q.rank, q.epoch);
    }
}

__global__ void __launch_bounds__(kFinalizeThreads)
laser_probe_reduce_kernel(const __grid_constant__ ReduceParams q) {
    const FinalizeParams& p = q.f;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    ptx::pdl_launch_dependents();
    ptx::pdl_wait();
    const int n = blockIdx.x * kFinalizeWarps + warp;
    const int n_valid = (p.R > 0) ? min(max(__ldg(p.req_offsets + p.R), 0), p.n_alloc) : 0;
    const RunPlan rp = resolve_plan(p.pd);
    if (n >= p.n_alloc) return;
    reduce_row(q, n, n_valid, rp.lay, lane);
}

// After the reduce kernel (stream order: its stores, remote ones included, have been performed):
// publish `epoch` in slot [rank] of every GPU's flag array with a system-scope release store.
__global__ void laser_probe_signal_kernel(const ReduceParams q) {
    publish_epoch(q, threadIdx.x);
}

// Host-buffer entry points: `hidden` in pinned, device-mapped host memory is pulled over PCIe by this
// kernel instead of a copy-engine transfer, so that the copy is a link of the same programmatic
// dependent launch chain as the probe kernels: its CTAs (no shared memory, few registers) become
// resident beside the previous call's fused CTAs and read their share of the rows into registers
// while that call is still running; only the stores into the staging buffer wait for it.
constexpr int kStageThreads = 256;
constexpr int kStageInFlight = 8;     // 16-byte loads per thread ahead of the wait
__global__ void __launch_bounds__(kStageThreads)
laser_probe_stage_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst, int64_t n16) {
    ptx::pdl_launch_dependents();
    const int64_t tid = static_cast<int64_t>(blockIdx.x) * kStageThreads + threadIdx.x;
    const int64_t nthreads = static_cast<int64_t>(gridDim.x) * kStageThreads;
    uint4 v[kStageInFlight];
#pragma unroll
    for (int j = 0; j < kStageInFlight; ++j) {
        const int64_t i = tid + j * nthreads;
        v[j] = i < n16 ? ptx::ld_nc_v4(src + i) : make_uint4(0u, 0u, 0u, 0u);
    }
    ptx::pdl_wait();    // the kernel ahead may still be reading the staging buffer
#pragma unroll
    for (int j = 0; j < kStageInFlight; ++j) {
        const int64_t i = tid + j * nthreads;
        if (i < n16) dst[i] = v[j];
    }
    for (int64_t i = tid + kStageInFlight * nthreads; i < n16; i += nthreads) dst[i] = ptx::ld_nc_v4(src + i);
}

// laser_probe_pack_w: [V, d] row-major -> [ceil(d/64)][V][64] (K-block-major), 16 bytes per thread and step;
// columns past d are zero.  Reads are 128-byte runs per row, writes are fully contiguous.
__global__ void __launch_bounds__(256)
laser_probe_pack_w_kernel(const uint4* __restrict__ W, uint4* __restrict__ out, int V, int d, int k_blocks) {
    const int64_t total = static_cast<int64_t>(k_blocks) * V * 8;     // 16-byte chunks of the packed buffer
    const int d16 = d >> 3;                                           // 16-byte chunks per row of W
    for (int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x; i < total;
         i += static_cast<int64_t>(gridDim.x) * blockDim.x) {
        const int c = static_cast<int>(i & 7);
        const int64_t r = i >> 3;                 // kb * V + v
        const int kb = static_cast<int>(r / V), v = static_cast<int>(r - static_cast<int64_t>(kb) * V);
        const int col16 = kb * 8 + c;
        out[i] = col16 < d16 ? W[static_cast<int64_t>(v) * d16 + col16] : make_uint4(0u, 0u, 0u, 0u);
    }
}

// LASER_DEBUG=1: the documented precondition on req_offsets (non-decreasing, [0] == 0, [R] <= N),
// checked on the device by one warp ahead of the probe; a violation traps (the caller sees a CUDA
// error at the next synchronisation) instead of silently reading other requests' rows.
__global__ void laser_probe_validate_kernel(const int32_t* req_offsets, int R, int N) {
    bool bad = false;
    for (int r = threadIdx.x; r <= R; r += 32) {
        const int v = req_offsets[r];
        if (r == 0 && v != 0) bad = true;
        if (r > 0 && v < req_offsets[r - 1]) bad = true;
        if (v < 0 || v > N) bad = true;
    }
    if (__any_sync(0xffffffffu, bad)) {
        if (threadIdx.x == 0) printf("laser_probe: req_offsets violates the precondition (non-decreasing, [0]==0, [R]<=N)\n");
        __trap();
    }
}

// ---------------------------------------------------------------------------------- fused kernel
// What the tail of the fused kernel does once every CTA's records are in the workspace.
//   kind 0: nothing (a second kernel follows: LASER_TAIL_SEPARATE)
//   kind 1: merge + a3-a5 (q.f), finalizer i takes requests i, i + F, ... with F = min(grid, R, kMaxFinalizers)
//   kind 2: vocabulary-parallel reduce (q): CTA b takes rows, the last CTA to finish publishes the epoch
// ctl: four device words owned by the library (never the caller's workspace):
//   ctl[0] counts CTA arrivals and only ever grows (wrap-safe compares); ctl[1] is the count at which
//   the current call started ("base"): every CTA reads it before it counts itself in, the LAST
//   arrival advances it by gridDim.x, so nothing is reset and no tail CTA reports back.  ctl[2]
//   (kind 2 only) counts tail CTAs whose rows have been pushed; the last one publishes the epoch and
//   clears it.  Calls that share a ctl slot must be stream-ordered (one handle = one slot).
#ifdef LASER_TIMELINE
// Debug build only (never the shipped library): per-CTA globaltimer stamps of the last 8 calls.
__device__ unsigned long long g_timeline[8][160][8];
__device__ __forceinline__ unsigned long long tl_now() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
#define LASER_TL(slot, ev, tid) do { if (threadIdx.x == (tid)) g_timeline[(slot) & 7][blockIdx.x][(ev)] = tl_now(); } while (0)
#else
#define LASER_TL(slot, ev, tid) do { } while (0)
#endif

struct TailParams {
    int32_t tl_slot;
    int32_t kind;
    uint32_t* ctl;
    ReduceParams q;
};

// Who takes part in a call's tail (decided per kernel, uniformly over its CTAs).
//   count_total  CTAs (of all fused kernels of the call) that count themselves in: the arrival target
//   fin_mode     0: the LAST F arrivals finalize (they have the least to wait for; fixed finalizers would
//                   spin for tens of microseconds in overlap mode);  1: CTAs [0, F) of this kernel
//                   finalize;  2: this kernel's CTAs only count themselves in;  -1: no tail here
//   part         CTAs of this kernel that take part (blockIdx.x < part): bounds F, strides the padding rows
struct TailRole {
    int count_total, fin_mode, part;
};
// Mixed schedule (pd.kind 2): only CTAs with work count.  Pair items only / single-CTA tiles only: the
// kernel that has the work runs the whole tail like a call with one fused kernel, the other stays out
// of it.  Both parts busy: the busy CTAs of both kernels count themselves in and the first F busy CTAs
// of the PAIR kernel finalize - it is launched behind the single-CTA kernel, so every CTA it waits
// for is resident or done (a dependent grid starts only when all CTAs of the grid ahead have
// started), while the single-CTA kernel never waits for anything launched after it: a tool that
// serialises the two kernels only costs time.  No row at all (req_offsets[R] == 0): every CTA of the
// pair kernel takes part, so that conf = 0 / exit = 0 / the padding marks are written.
__device__ __forceinline__ TailRole mixed_tail_role(const MixedPlan& mp, int role, int grid) {
    const int busy_pair = mp.k_pair > 0 ? 2 * mp.u_pair : 0;
    const int busy_single = mp.j_single > 0 ? mp.u_tail : 0;
    if (busy_pair + busy_single == 0) return role == 1 ? TailRole{grid, 0, grid} : TailRole{0, -1, 0};
    if (busy_single == 0) return role == 1 ? TailRole{busy_pair, 0, busy_pair} : TailRole{0, -1, 0};
    if (busy_pair == 0) return role == 2 ? TailRole{busy_single, 0, busy_single} : TailRole{0, -1, 0};
    return role == 1 ? TailRole{busy_pair + busy_single, 1, busy_pair} : TailRole{busy_pair + busy_single, 2, busy_single};
}

// The tail, run by the four epilogue warps (threads [kTailThread0, kTailThread0 + 128)) of every CTA
// that takes part (TailRole) once the CTA's records - if it had any to write - are stored: the CTA
// counts itself in, and the CTAs chosen as finalizers wait for the count to reach base + count_total
// and run merge + a3-a5 (kind 1) or the shard reduce (kind 2).
// base: ctl[1] as read by thread kTailThread0 when base_known (the call ahead, which may share the slot,
// had completed); otherwise it is read here.  cached: off_c / tau_c hold {req_offsets, tau} of every request.
__device__ __forceinline__ void fused_tail(const FusedParams& p, const TailParams& t, const RunPlan& rp,
                                           const TailRole tr, uint32_t base, bool base_known, bool cached,
                                           const int* off_c, const float* tau_c, float* warp_acc) {
    if (tr.fin_mode < 0 || static_cast<int>(blockIdx.x) >= tr.part) return;
    if (p.role != 1) ptx::pdl_wait();   // outputs are written below (a CTA without work items has not waited yet)
    const int tid = threadIdx.x - kTailThread0, tw = tid >> 5;
    constexpr int kTW = kEpilogueThreads / 32;
    const FinalizeParams& f = t.q.f;
    // At most kMaxFinalizers CTAs of a call ever spin on the arrival count.  A finalizer holds its SM while
    // it waits for CTAs that may not be resident yet (grids of other streams can be interleaved with this
    // one); were every CTA a finalizer, two such calls could each hold part of the SMs and wait for CTAs
    // that have nowhere to run.  With the cap, 148 - 32 k SMs stay free for the CTAs still to come when k
    // calls are in their tails at once (include/laser_probe.h: up to four fused-tail calls in flight).
    const int F = min((t.kind == 1) ? min(tr.part, f.R) : min(tr.part, (f.n_alloc + kTW - 1) / kTW), kMaxFinalizers);
    // scratch: bytes [192, 232) of the barrier block
    volatile uint32_t* tk = reinterpret_cast<volatile uint32_t*>(warp_acc + kMaxTailWarps);
    group_sync<1, kEpilogueThreads>();   // every record store of this CTA is ordered before the count
    if (tid == 0) {
        if (!base_known) base = ptx::ld_relaxed_gpu_u32(t.ctl + 1);   // overlap: the call ahead is complete only now
        const uint32_t target = base + static_cast<uint32_t>(tr.count_total);
        LASER_TL(t.tl_slot, 4, kTailThread0);
        const uint32_t mine = ptx::atom_add_acq_rel_gpu_u32(t.ctl, 1u) + 1u;
        if (mine == target) t.ctl[1] = target;   // last arrival: every CTA that counts has read `base`
        tk[0] = mine; tk[1] = target;
    }
    if (tr.fin_mode == 2) return;        // counted in, nothing else
    group_sync<1, kEpilogueThreads>();
    const uint32_t mine = tk[0], target = tk[1];
    const int behind = static_cast<int>(target - mine);    // CTAs still to arrive
    int fi;             // finalizer index 0 .. F-1, or -1
    if (tr.fin_mode == 1) fi = static_cast<int>(blockIdx.x) < F ? static_cast<int>(blockIdx.x) : -1;
    else fi = behind < F ? F - 1 - behind : -1;     // the last arrival is F-1
    const int pad_first = blockIdx.x * kEpilogueThreads + tid, pad_step = tr.part * kEpilogueThreads;
    if (fi < 0) {
        // not a finalizer: padding rows do not depend on anybody's records
        if (t.kind == 1) mark_padding_rows(f, pad_first, pad_step);
        return;
    }
    if (behind > 0) {
        if ((tid & 31) == 0) {
            const long long t0 = clock64();
            while (static_cast<int32_t>(ptx::ld_acquire_gpu_u32(t.ctl) - target) < 0) {
                // every CTA that counts is resident or becomes resident as others exit (grid <= SMs);
                // a wait of seconds means the device cannot hold the grid: trap
                if (clock64() - t0 > 8000000000LL) __trap();
            }
        }
        __syncwarp();
    }   // (the last arrival's own acq_rel count has acquired everybody's records)
    LASER_TL(t.tl_slot, 5, kTailThread0);
    if (t.kind == 1) {
        for (int r = fi; r < f.R; r += F) {
            const int rb = cached ? off_c[r] : __ldg(f.req_offsets + r);
            const int re = cached ? off_c[r + 1] : __ldg(f.req_offsets + r + 1);
            float tau = 0.f;
            if (tid == kFinalThread) tau = cached ? tau_c[r] : tau_eval(__ldg(f.load + r), f.tau);
            finalize_request<1, kEpilogueThreads>(f, tid, r, rb, re, tau, rp.lay, warp_acc);
            if (r == fi) LASER_TL(t.tl_slot, 6, kTailThread0);
        }
        mark_padding_rows(f, pad_first, pad_step);
    } else {
        const int n_valid = (f.R > 0) ? min(max(__ldg(f.req_offsets + f.R), 0), f.n_alloc) : 0;
        for (int n = fi * kTW + tw; n < f.n_alloc; n += F * kTW) reduce_row(t.q, n, n_valid, rp.lay, tid & 31);
        __threadfence_system();   // remote (peer) stores of this thread are performed before the count below
        group_sync<1, kEpilogueThreads>();
        if (tid < 32) {
            uint32_t last = 0;
            if (tid == 0) {
                last = (ptx::atom_add_acq_rel_gpu_u32(t.ctl + 2, 1u) == static_cast<uint32_t>(F - 1)) ? 1u : 0u;
                if (last) t.ctl[2] = 0u;
            }
            last = __shfl_sync(0xffffffffu, last, 0);
            if (last) publish_epoch(t.q, tid);   // every tail CTA's rows are on every GPU
        }
    }
}

// kPair = false: one CTA per SM, tcgen05 cta_group::1, a work item is (128 token rows, vocab split).
// kPair = true : clusters of two CTAs (the two SMs of a TPC), tcgen05 cta_group::2: one M = 256 MMA
//                spans both CTAs.  A work item is (256 token rows, vocab split); CTA `rank` of the pair
//                stages its own 128 token rows (A) and its own half of the vocabulary tile (B rows
//                [rank*BN/2, +BN/2)), so each W byte enters the pair's shared memory once instead of
//                once per 128-row token tile; the accumulator of CTA `rank` holds rows
//                [rank*128, +128) x all BN columns, and the epilogue is the same as in single mode.
//                Only the leader (rank 0) issues MMAs; its full barriers collect the TMA bytes of
//                both CTAs, its commits are multicast to both CTAs' barriers, and the epilogue warps
//                of both CTAs release the accumulator on the leader's tmem-empty barrier.
template <bool kPair>
__global__ void __launch_bounds__(kFusedThreads, 1)
laser_probe_fused_kernel(const __grid_constant__ CUtensorMap tmap_hidden,
                         const __grid_constant__ CUtensorMap tmap_w, const __grid_constant__ FusedParams p,
                         const __grid_constant__ TailParams t) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = ptx::smem_u32(smem_raw);
    const uint32_t smem = (raw + 1023u) & ~1023u;  // SWIZZLE_128B tiles need 1024-byte alignment
    const uint32_t bars = smem + static_cast<uint32_t>(p.stages) * p.stage_bytes;
    // barrier block: full[8] | empty[8] | tmem_full[2] | tmem_empty[2] | tmem base address (u32)
    auto full_bar = [&](int s) { return bars + 8u * s; };
    auto empty_bar = [&](int s) { return bars + 64u + 8u * s; };
    auto tfull_bar = [&](int b) { return bars + 128u + 8u * b; };
    auto tempty_bar = [&](int b) { return bars + 144u + 8u * b; };
    const uint32_t tmem_slot = bars + 160u;
    volatile uint32_t* tmem_slot_ptr =
        reinterpret_cast<volatile uint32_t*>(smem_raw + (smem - raw) + p.stages * p.stage_bytes + 160u);

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    LASER_TL(t.tl_slot, 0, 0);    // kernel entry
    const uint32_t rank = kPair ? ptx::cluster_ctarank() : 0u;   // 0 = leader
    const int unit = kPair ? (blockIdx.x >> 1) : blockIdx.x;     // CTA (single) or CTA pair
    const int units = kPair ? (gridDim.x >> 1) : gridDim.x;
    constexpr int kRowsPerItem = kPair ? 2 * kTileM : kTileM;
    constexpr int kEpiArrivals = kPair ? 8 : 4;                  // one per epilogue warp (of both CTAs)

    const int BN = p.tile_n;
    const int b_rows = kPair ? (BN >> 1) : BN;   // W rows this CTA stages per tile
    const int total_tiles = p.total_tiles;
    // static plan (pd.kind == 0); decided on the device further down otherwise
    int m_items = p.pd.m_tiles, S = p.pd.splits, units_run = units;
    int work_items = m_items * S;
    int row0 = 0;          // first token row of this kernel's items
    int64_t rec0 = 0;      // first workspace record of this kernel's region
    const bool static_plan = p.pd.kind == 0;
    RunPlan rp{};
    TailRole tr{p.grid_total, 0, static_cast<int>(gridDim.x)};   // one fused kernel: every CTA takes part
    if (p.pd.kind == 2) {
        // Mixed schedule: which part takes what is looked up before anything is set up, so that the
        // CTAs a part does not need (all of them, for the single-CTA kernel of an even dense batch)
        // leave within a microsecond or two.  The single-CTA kernel (role 2) orders the whole call
        // against the kernel ahead - it waits, THEN lets the pair kernel in, which never has to wait.
        if (p.role == 2) ptx::pdl_wait();
        rp = resolve_plan(p.pd);
        if (p.role == 2) ptx::pdl_launch_dependents();
        if (kPair) {             // pair part: k_pair items of 256 rows on u_pair pairs
            m_items = rp.mp.k_pair; S = rp.mp.S_pair; units_run = rp.mp.u_pair;
        } else {                 // the 128-row tiles behind the pair items on u_tail single CTAs
            m_items = rp.mp.j_single; S = rp.mp.S_tail; units_run = rp.mp.u_tail;
            row0 = 2 * kTileM * rp.mp.k_pair;
            rec0 = static_cast<int64_t>(row0) * rp.mp.S_pair;
        }
        tr = mixed_tail_role(rp.mp, p.role, gridDim.x);
        if (m_items == 0 || unit >= units_run) {
            // nothing to compute for this CTA.  It takes part in a fused tail only when no CTA of the
            // call has anything to compute (mixed_tail_role), and it completes only after the kernel
            // ahead of it has (completion of the pair kernel then implies completion of the whole call).
            if (p.role != 2) ptx::pdl_launch_dependents();
            if (t.kind != 0 && warp >= 2) {
                float* scratch = reinterpret_cast<float*>(smem_raw + (smem - raw) + p.stages * p.stage_bytes + 192u);
                fused_tail(p, t, rp, tr, 0u, false, false, nullptr, nullptr, scratch);
            }
            ptx::pdl_wait();
            return;
        }
        work_items = m_items * S;
    }

    // W ahead of the wait (strict mode, static plan): the producer requests the W boxes of its first
    // `stages` pipeline slots - and asks L2 for the boxes of the `stages` slots after those - before
    // griddepcontrol.wait, so that the head of the W stream overlaps whatever the kernel ahead of this
    // one still has to finish.  W is model weight: the kernel ahead never writes it (documented in
    // include/laser_probe.h).  The hidden boxes of those slots follow after the wait.
    int pre = 0;
    auto preissue_w = [&]() {
        if (!(p.early_w && static_plan && unit < work_items)) return;
        const uint32_t full0 = kPair ? ptx::mapa(full_bar(0), 0u) : full_bar(0);
        int tile = unit / m_items, kb = 0;
        for (int slot = 0; slot < p.stages + p.prefetch_slots && tile < total_tiles; ++slot) {
            if (ptx::elect_one()) {
                const int b_row = tile * BN + static_cast<int>(rank) * b_rows;
                if (slot < p.stages) {
                    const uint32_t sb = smem + static_cast<uint32_t>(slot) * p.stage_bytes + kABytes;
                    const uint32_t fb = full0 + 8u * slot;
                    if constexpr (kPair) {
                        if (rank == 0) ptx::mbar_arrive_expect_tx(full_bar(slot), 2u * p.tx_bytes);
                        ptx::tma_load_2d_pair(sb, &tmap_w, fb, w_c0(p, kb), w_c1(p, kb, b_row), p.w_policy);
                    } else {
                        ptx::mbar_arrive_expect_tx(fb, p.tx_bytes);
                        ptx::tma_load_2d(sb, &tmap_w, fb, w_c0(p, kb), w_c1(p, kb, b_row), p.w_policy);
                    }
                } else {
                    ptx::tma_prefetch_2d(&tmap_w, w_c0(p, kb), w_c1(p, kb, b_row));
                }
            }
            __syncwarp();
            if (slot < p.stages) ++pre;
            if (++kb == p.k_blocks) { kb = 0; tile += S; }
        }
    };

    if (warp == 0) {
        if (lane == 0) {
            ptx::prefetch_tensormap(&tmap_hidden);
            ptx::prefetch_tensormap(&tmap_w);
            for (int s = 0; s < p.stages; ++s) {
                ptx::mbar_init(full_bar(s), 1);
                ptx::mbar_init(empty_bar(s), 1);
            }
            for (int b = 0; b < 2; ++b) {
                ptx::mbar_init(tfull_bar(b), 1);
                ptx::mbar_init(tempty_bar(b), kEpiArrivals);
            }
            ptx::fence_mbar_init();
        }
        __syncwarp();
        // single CTA: its own barriers are all the loads need - do not wait for the TMEM allocation
        if constexpr (!kPair) preissue_w();
    }
    if (warp == 1) {
        ptx::tmem_alloc_t<kPair>(tmem_slot, kTmemCols);
        ptx::tmem_relinquish_t<kPair>();
    }
    ptx::tc_fence_before();
    if constexpr (kPair) ptx::cluster_sync();   // the peer's barriers exist before anything remote
    else __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    // Programmatic dependent launch: whatever follows in the stream may become resident on the SMs
    // this grid vacates; it must itself wait (griddepcontrol.wait) before it touches our outputs.
    // Role 2 (the first kernel of a mixed call) orders the whole call against the kernel ahead: it
    // waits first and only then lets the pair kernel (role 1) in, which therefore never has to wait.
    if (p.pd.kind != 2 || p.role == 1) ptx::pdl_launch_dependents();
    if constexpr (kPair) { if (warp == 0) preissue_w(); }
    LASER_TL(t.tl_slot, 1, 0);    // prologue + W pre-issue done

    // Strict: every read of hidden / req_offsets / token_ids below happens after the kernel ahead of
    // this one in the stream has completed.  Overlap: only the stores wait (further down).
    if (p.wait_first && p.role == 0) ptx::pdl_wait();
    LASER_TL(t.tl_slot, 2, 0);    // strict wait passed
    // tail bookkeeping: the arrival count this call starts from (strict: read here, long before it is
    // needed; the call ahead, which may share the slot, has completed)
    uint32_t base = 0;
    const bool base_early = p.wait_first || p.role != 0;   // the call ahead (same slot) has completed by now
    if (threadIdx.x == kTailThread0 && t.kind != 0 && base_early) base = ptx::ld_relaxed_gpu_u32(t.ctl + 1);
    // a4 ahead of time: {req_offsets, tau(load)} of every request into the shared-memory cache behind
    // the barrier block (any CTA may turn out to be one of the last to arrive)
    int* off_c = reinterpret_cast<int*>(smem_raw + (smem - raw) + p.stages * p.stage_bytes + 256u);
    float* tau_c = reinterpret_cast<float*>(off_c + p.tail_cache + 1);
    const bool cached = t.kind == 1 && t.q.f.R <= p.tail_cache;
    if (cached && warp >= 2) {
        const FinalizeParams& f = t.q.f;
        for (int i = threadIdx.x - kTailThread0; i <= f.R; i += kEpilogueThreads) {
            off_c[i] = __ldg(f.req_offsets + i);
            if (i < f.R) tau_c[i] = tau_eval(__ldg(f.load + i), f.tau);
        }
    }

    if (static_plan) {
        rp.m_items = m_items; rp.S = S;
        rp.lay = RecLayout{0x7fffffff, S, S};
    } else if (p.pd.kind == 1) {
        rp = resolve_plan(p.pd);
        m_items = rp.m_items; S = rp.S;
        work_items = m_items * S;
        if (m_items == 0) { m_items = 1; work_items = 0; }
    }
    // split sp owns vocabulary tiles sp, sp + S, sp + 2S, ... (ascending: ties keep the lowest index)

    if (warp == 0) {
        // ===================================================================== TMA producer
        // Converged warp, one elected lane issues (see the MMA issuer).
        const int k_blocks = p.k_blocks, stages = p.stages;
        const uint32_t full0 = kPair ? ptx::mapa(full_bar(0), 0u) : full_bar(0);  // leader's barriers
        int stage = 0;
        uint32_t phase = 0;
        for (int w = unit; w < work_items; w += units_run) {
            const int mt = w % m_items, sp = w / m_items;
            const int a_row = row0 + mt * kRowsPerItem + static_cast<int>(rank) * kTileM;
            for (int tile = sp; tile < total_tiles; tile += S) {
                const int b_row = tile * BN + static_cast<int>(rank) * b_rows;
                for (int kb = 0; kb < k_blocks; ++kb) {
                    const uint32_t sa = smem + static_cast<uint32_t>(stage) * p.stage_bytes;
                    const uint32_t fb = full0 + 8u * stage;
                    if (pre > 0) {
                        // slot whose W box (and expected byte count) went out ahead of the wait
                        --pre;
                        if (ptx::elect_one()) {
                            if constexpr (kPair)
                                ptx::tma_load_2d_pair(sa, &tmap_hidden, fb, kb * kBlockK, a_row, ptx::kEvictLast);
                            else
                                ptx::tma_load_2d(sa, &tmap_hidden, fb, kb * kBlockK, a_row, ptx::kEvictLast);
                        }
                    } else {
                        ptx::mbar_wait(empty_bar(stage), phase ^ 1u);
                        if (ptx::elect_one()) {
                            if constexpr (kPair) {
                                // both CTAs' bytes complete on the leader's barrier
                                if (rank == 0) ptx::mbar_arrive_expect_tx(full_bar(stage), 2u * p.tx_bytes);
                                ptx::tma_load_2d_pair(sa, &tmap_hidden, fb, kb * kBlockK, a_row, ptx::kEvictLast);
                                ptx::tma_load_2d_pair(sa + kABytes, &tmap_w, fb, w_c0(p, kb), w_c1(p, kb, b_row), p.w_policy);
                            } else {
                                ptx::mbar_arrive_expect_tx(fb, p.tx_bytes);
                                ptx::tma_load_2d(sa, &tmap_hidden, fb, kb * kBlockK, a_row, ptx::kEvictLast);
                                ptx::tma_load_2d(sa + kABytes, &tmap_w, fb, w_c0(p, kb), w_c1(p, kb, b_row), p.w_policy);
                            }
                        }
                    }
                    __syncwarp();
                    if (++stage == stages) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================================================================== MMA issuer
        // The whole warp walks the loop converged (every lane polls the barriers); one elected lane
        // issues.  Descriptors advance by additions only: +2 per UMMA_K step inside the 128-byte
        // swizzle row, +stage_bytes/16 per pipeline stage.
        if (rank == 0) {
            const uint32_t idesc = make_idesc_bf16(static_cast<uint32_t>(BN), kRowsPerItem);
            const uint64_t a_desc0 = make_smem_desc_sw128(smem);
            const uint64_t b_desc0 = make_smem_desc_sw128(smem + kABytes);
            const uint32_t stage_step = p.stage_bytes >> 4;
            const int k_blocks = p.k_blocks, stages = p.stages;
            int stage = 0;
            uint32_t phase = 0, acc = 0, desc_off = 0;
            for (int w = unit; w < work_items; w += units_run) {
                for (int tile = w / m_items; tile < total_tiles; tile += S, ++acc) {
                    const uint32_t buf = acc & 1u, aphase = (acc >> 1) & 1u;
                    // epilogue (of both CTAs in pair mode) drained this buffer
                    if constexpr (kPair) ptx::mbar_wait_cluster(tempty_bar(buf), aphase ^ 1u);
                    else ptx::mbar_wait(tempty_bar(buf), aphase ^ 1u);
                    ptx::tc_fence_after();
                    const uint32_t d_tmem = tmem_base + buf * kMaxTileN;
                    for (int kb = 0; kb < k_blocks; ++kb) {
                        ptx::mbar_wait(full_bar(stage), phase);  // TMA bytes have landed
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
                            const uint64_t a_desc = a_desc0 + desc_off;
                            const uint64_t b_desc = b_desc0 + desc_off;
                            ptx::umma_bf16_t<kPair>(d_tmem, a_desc, b_desc, idesc, kb != 0);
                            ptx::umma_bf16_t<kPair>(d_tmem, a_desc + 2u, b_desc + 2u, idesc, 1u);
                            ptx::umma_bf16_t<kPair>(d_tmem, a_desc + 4u, b_desc + 4u, idesc, 1u);
                            ptx::umma_bf16_t<kPair>(d_tmem, a_desc + 6u, b_desc + 6u, idesc, 1u);
                            ptx::umma_commit_t<kPair>(empty_bar(stage));  // frees the stage when the MMAs retire
                            if (kb == k_blocks - 1)
                                ptx::umma_commit_t<kPair>(tfull_bar(buf));  // accumulator complete -> epilogue
                        }
                        __syncwarp();
                        desc_off += stage_step;
                        if (++stage == stages) { stage = 0; phase ^= 1u; desc_off = 0; }
                    }
                }
            }
        }
    } else {
        // ===================================================================== epilogue (4 warps)
        const int q = warp & 3;  // a warp may only touch TMEM lanes [32*(warp%4), +32)
        const int row = static_cast<int>(rank) * kTileM + q * 32 + lane;
        const uint32_t lane_addr = static_cast<uint32_t>(q * 32) << 16;
        uint32_t acc = 0;
        for (int w = unit; w < work_items; w += units_run) {
            const int mt = w % m_items, sp = w / m_items;
            float m = -CUDART_INF_F, s = 0.f, lt = -CUDART_INF_F;
            int a = -1, tok = -1;
            if (p.token_ids != nullptr) {
                const int n = row0 + mt * kRowsPerItem + row;
                if (n < p.n_alloc) {
                    const int tk = __ldg(p.token_ids + n) - p.v_offset;
                    tok = (tk >= 0 && tk < p.V) ? tk : -1;   // not in this (shard of the) vocabulary
                }
            }
            for (int tile = sp; tile < total_tiles; tile += S, ++acc) {
                const uint32_t buf = acc & 1u, aphase = (acc >> 1) & 1u;
                ptx::mbar_wait(tfull_bar(buf), aphase);
                ptx::tc_fence_after();
                const uint32_t taddr = tmem_base + lane_addr + buf * kMaxTileN;
                const int vt = tile * BN;
                int c = 0;
                for (; c + 32 <= BN && vt + c < p.V; c += 32) {
                    uint32_t r[32];
                    ptx::tmem_ld_x32(taddr + c, r);
                    ptx::tmem_wait_ld();
                    fold_columns<32>(r, vt + c, p.V, m, a, s, tok, lt);
                }
                // tile_n is a multiple of 16: at most one 16-column tail chunk
                if (c + 16 == BN && vt + c < p.V) {
                    uint32_t r[16];
                    ptx::tmem_ld_x16(taddr + c, r);
                    ptx::tmem_wait_ld();
                    fold_columns<16>(r, vt + c, p.V, m, a, s, tok, lt);
                }
                // all of this warp's TMEM reads have completed (wait::ld): one arrival per warp
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    if constexpr (kPair) ptx::mbar_arrive_cluster(ptx::mapa(tempty_bar(buf), 0u));
                    else ptx::mbar_arrive(tempty_bar(buf));
                }
            }
            // packed row-major over splits: the merge reads a row's partials as contiguous 16-byte
            // records (coalesced); the scattered 16-byte stores here are fire-and-forget
            const int64_t o = rec0 + (static_cast<int64_t>(mt) * kRowsPerItem + row) * S + sp;
            // overlap mode: the previous call's tail may still be reading the workspace.  (Role 1 must
            // not wait: the kernel ahead of it is its own call's role-2 kernel, ordered already.)
            if (p.role != 1) ptx::pdl_wait();
            p.ws[o] = make_float4(m, s, __int_as_float(a), lt);
        }
        LASER_TL(t.tl_slot, 3, kTailThread0);   // last record stored
        // This warp is done with TMEM and the pipeline: tell the teardown below (TMEM deallocation by
        // warp 1) without waiting for it - the tail that follows needs neither.
        ptx::tc_fence_before();
        if constexpr (kPair) ptx::cluster_arrive();
        else asm volatile("bar.arrive 2, %0;" ::"n"(kFusedThreads) : "memory");

        // ================================================================= tail (epilogue warps only)
        // The four epilogue warps count this CTA in as soon as their records are stored - the producer
        // and MMA warps go straight to the teardown - and the LAST F CTAs to arrive run merge + a3-a5
        // (kind 1) or the shard reduce (kind 2): they are the ones with the least to wait for.
        if (t.kind != 0) {
            float* scratch = reinterpret_cast<float*>(smem_raw + (smem - raw) + p.stages * p.stage_bytes + 192u);
            fused_tail(p, t, rp, tr, base, base_early, cached, off_c, tau_c, scratch);
        }
    }

    // ------------------------------------------------------------------------- teardown
    __syncwarp();   // reconverge the warps whose lane 0 ran a role loop
    LASER_TL(t.tl_slot, 7, 0);    // producer done issuing
    // No CTA (not even one without work) completes before the kernel ahead of it in the stream has:
    // completion of this grid then implies completion of everything before it, as stream order demands.
    ptx::pdl_wait();
    if (warp >= 2) {
        // epilogue warps arrived before their tail; the cluster barrier wants every arrival waited for
        if constexpr (kPair) ptx::cluster_wait();
        return;
    }
    ptx::tc_fence_before();
    // all epilogue warps (of both CTAs of a pair: the peer may still read this CTA's shared memory /
    // TMEM) have finished with TMEM
    if constexpr (kPair) ptx::cluster_sync();
    else asm volatile("bar.sync 2, %0;" ::"n"(kFusedThreads) : "memory");
    if (warp == 1) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc_t<kPair>(tmem_base, kTmemCols);
    }
}

}  // namespace laser
