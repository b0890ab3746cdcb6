// probe_kernels.cuh — the two kernels of the LASER confidence probe (sm_100a).
//
//  laser_probe_fused_kernel   a1 + a2 of include/laser_probe.h: LM-head projection on tcgen05 tensor
//                             cores with the online-softmax statistics (max, lowest-index argmax,
//                             sum-exp) taken straight out of TMEM.  Logits never reach HBM.
//  laser_probe_finalize_kernel  merge of the per-split statistics (warp shuffles), a3 per-request
//                             aggregate, a4 threshold (Eq. 5 + clamp), a5 exit mask.
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
constexpr float kLog2e = 1.4426950408889634f;

// How the vocabulary tiles are dealt to the execution units (CTAs, or CTA pairs) for `m_items` token
// items: deal the `total_tiles` tiles of tile_n rows to `splits` splits of at most `T` tiles each such
// that m_items * splits fills the units in whole rounds with the least work on the busiest unit.
// Shared by the host planner and both kernels: when a batch carries padding rows (req_offsets[R] <
// N) the kernels re-plan on the device for the token items that actually hold rows.
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

struct FusedParams {
    int32_t n_alloc, d, V;
    int32_t m_tiles, splits, tiles_per_split, tile_n, k_blocks, stages;
    int32_t work_items, n_pad;   // m_tiles counts items of 128 (single) / 256 (pair) token rows
    uint32_t tx_bytes;     // bytes TMA delivers per stage and CTA (hidden box + W box)
    uint32_t stage_bytes;  // shared-memory stride of a stage: kABytes + (W rows per CTA) * 128
    uint64_t w_policy;     // L2 eviction policy for the W stream
    float4* ws;            // [n_pad, splits] per (row, split): {max, sum exp(logit - max), argmax bits, token logit}
    // LASER_PROB_TOKEN: token_ids[n] - v_offset is the column of W whose logit is kept for row n
    // (nullptr: no token logit is tracked; v_offset = global vocabulary index of W's row 0).
    const int32_t* token_ids;
    int32_t v_offset;
    // Padding-aware re-planning (m_tiles > 1 only): token items at or beyond req_offsets[R] are
    // skipped and the vocabulary tiles are re-dealt over the remaining items; `splits` above stays
    // the record stride (the largest split count any item count can produce).
    const int32_t* req_offsets;
    int32_t R, total_tiles, units, replan;
    // 1: griddepcontrol.wait before the first global read (strict stream order for the inputs too);
    // 0: only the workspace stores wait (see laser_probe_set_overlap in include/laser_probe.h).
    int32_t wait_first;
};

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

// ---------------------------------------------------------------------------------- fused kernel
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
                         const __grid_constant__ CUtensorMap tmap_w, const FusedParams p) {
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
    const uint32_t rank = kPair ? ptx::cluster_ctarank() : 0u;   // 0 = leader
    const int unit = kPair ? (blockIdx.x >> 1) : blockIdx.x;     // CTA (single) or CTA pair
    const int units = kPair ? (gridDim.x >> 1) : gridDim.x;
    constexpr int kRowsPerItem = kPair ? 2 * kTileM : kTileM;
    constexpr int kEpiArrivals = kPair ? 8 : 4;                  // one per epilogue warp (of both CTAs)

    if (warp == 0 && lane == 0) {
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
    if (warp == 1) {
        ptx::tmem_alloc_t<kPair>(tmem_slot, kTmemCols);
        ptx::tmem_relinquish_t<kPair>();
    }
    ptx::tc_fence_before();
    if constexpr (kPair) ptx::cluster_sync();   // the peer's barriers exist before anything remote
    else __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    // Programmatic dependent launch.  wait_first (the library default, laser_probe_set_overlap(0)):
    // every global read below happens after the kernel ahead of this one in the stream has completed;
    // only the prologue above overlapped it.  Without it (overlap opted in): the only memory this
    // kernel shares with the kernel before it in a chain of probe calls (the previous call's finalize
    // kernel) is the workspace, so only the workspace stores (and the exit) wait for that kernel and
    // the W stream of this call overlaps the tail of the previous one.
    if (p.wait_first) ptx::pdl_wait();
    // Let the finalize kernel's CTAs become resident now (they block in griddepcontrol.wait).
    ptx::pdl_launch_dependents();

    int m_items = p.m_tiles, work_items = p.work_items;
    const int BN = p.tile_n;
    const int b_rows = kPair ? (BN >> 1) : BN;   // W rows this CTA stages per tile
    if (p.replan) {   // uniform across the grid: every thread reads the same word
        const int n_valid = min(max(__ldg(p.req_offsets + p.R), 0), p.n_alloc);
        m_items = (n_valid + kRowsPerItem - 1) / kRowsPerItem;
        if (m_items < p.m_tiles) {
            if (m_items > 0) {
                work_items = m_items * plan_splits(p.total_tiles, m_items, p.units).splits;
            } else {
                work_items = 0;
            }
        }
    }
    // split sp owns vocabulary tiles sp, sp + S, sp + 2S, ... (ascending: ties keep the lowest index)
    const int S = m_items > 0 ? work_items / m_items : 1;
    const int total_tiles = p.total_tiles;

    if (warp == 0) {
        // ===================================================================== TMA producer
        // Converged warp, one elected lane issues (see the MMA issuer).
        {
            const int k_blocks = p.k_blocks, stages = p.stages;
            const uint32_t full0 = kPair ? ptx::mapa(full_bar(0), 0u) : full_bar(0);  // leader's barriers
            int stage = 0;
            uint32_t phase = 0;
            for (int w = unit; w < work_items; w += units) {
                const int mt = w % m_items, sp = w / m_items;
                const int a_row = mt * kRowsPerItem + static_cast<int>(rank) * kTileM;
                for (int tile = sp; tile < total_tiles; tile += S) {
                    const int b_row = tile * BN + static_cast<int>(rank) * b_rows;
                    for (int kb = 0; kb < k_blocks; ++kb) {
                        ptx::mbar_wait(empty_bar(stage), phase ^ 1u);
                        if (ptx::elect_one()) {
                            const uint32_t sa = smem + static_cast<uint32_t>(stage) * p.stage_bytes;
                            const uint32_t fb = full0 + 8u * stage;
                            if constexpr (kPair) {
                                // both CTAs' bytes complete on the leader's barrier
                                if (rank == 0) ptx::mbar_arrive_expect_tx(full_bar(stage), 2u * p.tx_bytes);
                                ptx::tma_load_2d_pair(sa, &tmap_hidden, fb, kb * kBlockK, a_row, ptx::kEvictLast);
                                ptx::tma_load_2d_pair(sa + kABytes, &tmap_w, fb, kb * kBlockK, b_row, p.w_policy);
                            } else {
                                ptx::mbar_arrive_expect_tx(fb, p.tx_bytes);
                                ptx::tma_load_2d(sa, &tmap_hidden, fb, kb * kBlockK, a_row, ptx::kEvictLast);
                                ptx::tma_load_2d(sa + kABytes, &tmap_w, fb, kb * kBlockK, b_row, p.w_policy);
                            }
                        }
                        __syncwarp();
                        if (++stage == stages) { stage = 0; phase ^= 1u; }
                    }
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
            for (int w = unit; w < work_items; w += units) {
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
        for (int w = unit; w < work_items; w += units) {
            const int mt = w % m_items, sp = w / m_items;
            float m = -CUDART_INF_F, s = 0.f, lt = -CUDART_INF_F;
            int a = -1, tok = -1;
            if (p.token_ids != nullptr) {
                const int n = mt * kRowsPerItem + row;
                if (n < p.n_alloc) {
                    const int t = __ldg(p.token_ids + n) - p.v_offset;
                    tok = (t >= 0 && t < p.V) ? t : -1;   // not in this (shard of the) vocabulary
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
            // row-major over splits: the finalize kernel reads a row's partials as contiguous 16-byte
            // records (coalesced); the scattered 16-byte stores here are fire-and-forget
            const size_t o = (static_cast<size_t>(mt) * kRowsPerItem + row) * p.splits + sp;
            ptx::pdl_wait();   // the previous call's finalize kernel may still be reading the workspace
            p.ws[o] = make_float4(m, s, __int_as_float(a), lt);
        }
    }

    // ------------------------------------------------------------------------- teardown
    __syncwarp();   // reconverge the warps whose lane 0 ran a role loop
    // No CTA (not even one without work) completes before the kernel ahead of it in the stream has:
    // completion of this grid then implies completion of everything before it, as stream order demands.
    ptx::pdl_wait();
    ptx::tc_fence_before();
    if constexpr (kPair) ptx::cluster_sync();   // the peer may still read this CTA's shared memory / TMEM
    else __syncthreads();
    if (warp == 1) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc_t<kPair>(tmem_base, kTmemCols);
    }
}

// ---------------------------------------------------------------------------------- finalize
struct TauParamsDev {
    float lambda_base, beta, gamma, l_target, lambda_min, lambda_max;
};

// a4: Eq. 5 then the clamp.  Shared by the kernel and laser_tau_from_load.
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
    int32_t n_alloc, R, splits, n_pad, agg_mode;
    int32_t m_tiles, rows_per_item, total_tiles, units, replan;   // see FusedParams
    // record (n, sp) lives at ws[n * row_stride + sp * split_stride]:
    //   fused workspace [n_pad, splits]: row_stride = splits, split_stride = 1
    //   gathered shard statistics [G, N]: row_stride = 1, split_stride = N  (laser_probe_combine)
    int64_t row_stride, split_stride;
    int32_t prob_mode;            // 0: row maximum 1/S; 1: the row's token exp(l_tok - m)/S
    int32_t a_offset;             // added to every argmax (vocabulary shard offset; reduce kernel)
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

// (m,a,s,lt) (+) (m',a',s',lt'): commutative form - on equal maxima the smaller vocabulary index
// wins; at most one operand carries a finite token logit.
__device__ __forceinline__ void merge_stats(float& m, int& a, float& s, float& lt, float m2, int a2,
                                            float s2, float lt2) {
    const float M = fmaxf(m, m2);
    const int an = (m > m2) ? a : ((m2 > m) ? a2 : min(a, a2));
    const float e1 = (m == M) ? 1.f : ptx::ex2_approx((m - M) * kLog2e);
    const float e2 = (m2 == M) ? 1.f : ptx::ex2_approx((m2 - M) * kLog2e);
    s = s * e1 + s2 * e2;
    m = M;
    a = an;
    lt = fmaxf(lt, lt2);
}

constexpr int kFinalizeThreads = 256;
constexpr int kFinalizeWarps = kFinalizeThreads / 32;
constexpr int kMergeBatch = 5;  // partials a lane loads before it starts merging (148 splits: one batch)

// Merge the nsplit records of one row across a warp (lanes stride over the records, loads issued in
// batches so that they overlap; then shuffles).  Every lane returns the merged statistics.
__device__ __forceinline__ void merge_row(const float4* rec, int64_t split_stride, int nsplit, int lane,
                                          float& m, int& a, float& s, float& lt) {
    m = -CUDART_INF_F; s = 0.f; lt = -CUDART_INF_F;
    a = 0x7fffffff;
    for (int sp0 = lane; sp0 < nsplit; sp0 += 32 * kMergeBatch) {
        float4 v[kMergeBatch];
#pragma unroll
        for (int j = 0; j < kMergeBatch; ++j) {
            const int sp = sp0 + 32 * j;
            v[j] = sp < nsplit ? rec[sp * split_stride]
                               : make_float4(-CUDART_INF_F, 0.f, __int_as_float(0x7fffffff), -CUDART_INF_F);
        }
#pragma unroll
        for (int j = 0; j < kMergeBatch; ++j)
            merge_stats(m, a, s, lt, v[j].x, __float_as_int(v[j].z), v[j].y, v[j].w);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const float m2 = __shfl_xor_sync(0xffffffffu, m, off);
        const int a2 = __shfl_xor_sync(0xffffffffu, a, off);
        const float s2 = __shfl_xor_sync(0xffffffffu, s, off);
        const float l2 = __shfl_xor_sync(0xffffffffu, lt, off);
        merge_stats(m, a, s, lt, m2, a2, s2, l2);
    }
}

// Records per row the fused kernel wrote for this batch (device-side re-plan, see FusedParams).
__device__ __forceinline__ int records_per_row(const FinalizeParams& p) {
    int nsplit = p.splits;
    if (p.replan) {
        const int n_valid = min(max(__ldg(p.req_offsets + p.R), 0), p.n_alloc);
        const int m_items = (n_valid + p.rows_per_item - 1) / p.rows_per_item;
        if (m_items > 0) nsplit = plan_splits(p.total_tiles, min(m_items, p.m_tiles), p.units).splits;
    }
    return nsplit;
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

// Blocks [0, R): one request each.  A warp takes rows b+w, b+w+8, ...: its lanes stride over the
// records of the row, fold their own, then merge across the warp with shuffles.
// Blocks [R, R + ceil(n_alloc/256)): mark padding rows (n >= req_offsets[R]).
// Everything that does not depend on the fused kernel (offsets, load, threshold) is read before
// griddepcontrol.wait so that under programmatic dependent launch it overlaps the fused kernel.
// launch_dependents is issued first of all: the next call's fused kernel may then take every SM the
// current fused kernel vacates and run its prologue there; it still blocks in its own
// griddepcontrol.wait until this grid (hence, transitively, the current fused kernel) has completed.
__global__ void __launch_bounds__(kFinalizeThreads)
laser_probe_finalize_kernel(const FinalizeParams p) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    ptx::pdl_launch_dependents();
    if (static_cast<int>(blockIdx.x) >= p.R) {
        const int n = (blockIdx.x - p.R) * kFinalizeThreads + threadIdx.x;
        const int n_valid = (p.R > 0) ? __ldg(p.req_offsets + p.R) : 0;
        if (n < p.n_alloc && n >= n_valid) {   // outputs of padding rows: independent of the fused kernel
            p.out_argmax[n] = -1;
            if (p.out_pmax) p.out_pmax[n] = CUDART_NAN_F;
        }
        return;
    }
    __shared__ float warp_acc[kFinalizeWarps];
    const int r = blockIdx.x;
    const int b = __ldg(p.req_offsets + r), e = __ldg(p.req_offsets + r + 1);
    float tau = 0.f;
    if (threadIdx.x == 0) tau = tau_eval(__ldg(p.load + r), p.tau);   // a4
    const int nsplit = records_per_row(p);

    ptx::pdl_wait();  // all of the fused kernel's partials are visible after this
    if (p.wait_flags != nullptr) wait_peer_flags(p.wait_flags, nsplit, p.epoch);

    // running aggregate of this warp's rows: sum (mean), sum of logs (geomean), min
    float acc = (p.agg_mode == 2) ? CUDART_INF_F : 0.f;
    bool any_nan = false;
    for (int n = b + warp; n < e; n += kFinalizeWarps) {
        float m, s, lt;
        int a;
        merge_row(p.ws + static_cast<int64_t>(n) * p.row_stride, p.split_stride, nsplit, lane, m, a, s, lt);
        // s >= 1 up to the rounding of ex2.approx; a probability does not exceed 1.  NaN stays NaN.
        float prob;
        if (p.prob_mode == 0) {
            prob = (s == s) ? fminf(1.0f / s, 1.0f) : CUDART_NAN_F;
        } else {   // the row's token: exp(l_tok - m) / S; a token outside the vocabulary has l_tok = -inf -> 0
            prob = (s == s) ? fminf(ptx::ex2_approx((lt - m) * kLog2e) / s, 1.0f) : CUDART_NAN_F;
        }
        if (lane == 0) {
            p.out_argmax[n] = a;
            if (p.out_pmax) p.out_pmax[n] = prob;
        }
        any_nan |= (prob != prob);
        if (p.agg_mode == 0) acc += prob;
        else if (p.agg_mode == 1) acc += logf(prob);
        else acc = fminf(acc, prob);
    }
    if (p.agg_mode == 2 && any_nan) acc = CUDART_NAN_F;
    if (lane == 0) warp_acc[warp] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        const int len = e - b;
        float conf = 0.f;
        if (len > 0) {
            if (p.agg_mode == 2) {
                conf = warp_acc[0];
                bool nan = conf != conf;
                for (int w = 1; w < kFinalizeWarps; ++w) {
                    nan |= (warp_acc[w] != warp_acc[w]);
                    conf = fminf(conf, warp_acc[w]);
                }
                if (nan) conf = CUDART_NAN_F;
            } else {
                float t = 0.f;
                for (int w = 0; w < kFinalizeWarps; ++w) t += warp_acc[w];
                conf = t / static_cast<float>(len);
                if (p.agg_mode == 1) conf = expf(conf);
            }
        }
        p.out_conf[r] = conf;                  // a3
        p.out_exit[r] = (conf > tau) ? 1 : 0;  // a5: strict; NaN > tau is false
        if (p.out_tau) p.out_tau[r] = tau;
    }
}

// ---------------------------------------------------------------------------------- vocab-parallel
// laser_probe_partial: the fused kernel over one vocabulary SHARD, then this kernel: one warp per row
// merges the row's split records into a single record {m, S, argmax + v_offset, l_tok} and stores it
//   * to out_stats[n] (local), and
//   * when peers are given, to slot [rank, n] of every GPU's gathered buffer [G, N] through
//     peer-mapped pointers (NVLink stores; 16 bytes per row and peer) - the all-gather of the
//     statistics is done by the producer, no collective call.
// Rows n >= req_offsets[R] (padding) get the neutral record.
constexpr int kMaxPeers = 16;
struct ReduceParams {
    FinalizeParams f;          // ws, strides, replan fields, req_offsets, R, n_alloc, a_offset
    float4* out_stats;         // [n_alloc] or nullptr
    int32_t rank, world;       // world = 0: no peers
    float4* peer_stats[kMaxPeers];   // peer_stats[g] = base of GPU g's gathered buffer [world, n_alloc]
};

__global__ void __launch_bounds__(kFinalizeThreads)
laser_probe_reduce_kernel(const ReduceParams q) {
    const FinalizeParams& p = q.f;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    ptx::pdl_launch_dependents();
    const int n = blockIdx.x * kFinalizeWarps + warp;
    const int n_valid = (p.R > 0) ? min(max(__ldg(p.req_offsets + p.R), 0), p.n_alloc) : 0;
    const int nsplit = records_per_row(p);
    ptx::pdl_wait();
    if (n >= p.n_alloc) return;
    float m = -CUDART_INF_F, s = 0.f, lt = -CUDART_INF_F;
    int a = 0x7fffffff;
    if (n < n_valid) {
        merge_row(p.ws + static_cast<int64_t>(n) * p.row_stride, p.split_stride, nsplit, lane, m, a, s, lt);
        a += p.a_offset;
    }
    const float4 rec = make_float4(m, s, __int_as_float(a), lt);
    if (lane == 0 && q.out_stats) q.out_stats[n] = rec;
    if (lane < q.world) q.peer_stats[lane][static_cast<int64_t>(q.rank) * p.n_alloc + n] = rec;
}

// After the reduce kernel (stream order: its stores, remote ones included, have been performed):
// publish `epoch` in slot [rank] of every GPU's flag array with a system-scope release store.
struct SignalParams {
    int32_t rank, world;
    uint32_t epoch;
    uint32_t* peer_flags[kMaxPeers];   // peer_flags[g] = GPU g's flag array [world]
};
__global__ void laser_probe_signal_kernel(const SignalParams q) {
    const int g = threadIdx.x;
    if (g < q.world) {
        __threadfence_system();
        ptx::st_release_sys_u32(q.peer_flags[g] + q.rank, q.epoch);
    }
}

}  // namespace laser
