// flex_kernel.cuh — laser_probe_flex_kernel: a1 + a2 (+ the tail: merge, a3-a5) with the operands of the
// projection swapped (sm_100a, CTA pairs).
//
// laser_probe_fused_kernel puts the token rows on the MMA M axis, which tcgen05 fixes at 128 rows per CTA:
// a batch of 320 or 590 rows pays for 384 or 640-768.  Here the VOCABULARY is on M (a tile = 256 rows of
// W per CTA pair, 128 TMEM lanes per CTA) and the TOKENS are on N, which UMMA takes in steps of 16 up to
// 256: the valid rows are cut into C chunks of n_tok rows (a multiple of 16), so a batch pays for at most
// 15 rows of padding per chunk - decided on the device from req_offsets[R] through a table the host
// planned for every count of 16-row groups (PlanDesc kind 3).
//
// The accumulator of a (vocabulary tile, token chunk) therefore holds logits[v, n] with v on the TMEM
// lanes: the softmax axis runs ACROSS the threads of an epilogue warp.  Each warp turns its 32 x 32 block
// (32 vocabulary rows x 32 tokens) around through 4 KB of shared memory of its own (conflict-free XOR
// swizzle, __syncwarp only) and then every thread folds 32 ascending vocabulary columns of ONE token with
// the same fold_columns as the other kernel; a thread keeps the running (max, argmax, sum-exp) of up to 8
// tokens (one per 32-token group of the chunk).  At the end of a work item the four warps' statistics of
// a token (four vocabulary quarters) meet in the same shared memory and one record per (row, split, CTA)
// goes to the workspace: 2 S records per row, merged by the common tail.
//
// Everything else - TMA ring, elected issuers, double-buffered TMEM accumulators, programmatic dependent
// launch, the arrival-counting tail - is the CTA-pair form of laser_probe_fused_kernel.
#pragma once
#include "probe_kernels.cuh"

namespace laser {

constexpr int kFlexMaps = kFlexMaxTok / 16;        // hidden tensor maps: box of 8 * (i + 1) token rows
constexpr int kFlexXposeBytes = 4 * 32 * 32 * 4;   // four warps x (32 x 32 floats)
struct FlexMaps {
    CUtensorMap hid[kFlexMaps];
};

__global__ void __launch_bounds__(kFusedThreads, 1)
laser_probe_flex_kernel(const __grid_constant__ FlexMaps tm_hid, const __grid_constant__ CUtensorMap tmap_w,
                        const __grid_constant__ FusedParams p, const __grid_constant__ TailParams t) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = ptx::smem_u32(smem_raw);
    const uint32_t smem = (raw + 1023u) & ~1023u;
    uint8_t* const smem_gen = smem_raw + (smem - raw);
    const uint32_t ring_bytes = static_cast<uint32_t>(p.stages) * p.stage_bytes;
    // ring | transpose / record exchange (16 KB) | barrier block (256 B) | tail cache
    float* const xpose = reinterpret_cast<float*>(smem_gen + ring_bytes);
    const uint32_t bars = smem + ring_bytes + kFlexXposeBytes;
    uint8_t* const bars_gen = smem_gen + ring_bytes + kFlexXposeBytes;
    auto full_bar = [&](int s) { return bars + 8u * s; };
    auto empty_bar = [&](int s) { return bars + 64u + 8u * s; };
    auto tfull_bar = [&](int b) { return bars + 128u + 8u * b; };
    auto tempty_bar = [&](int b) { return bars + 144u + 8u * b; };
    const uint32_t tmem_slot = bars + 160u;
    volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(bars_gen + 160u);

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    LASER_TL(t.tl_slot, 0, 0);
    const uint32_t rank = ptx::cluster_ctarank();   // 0 = leader
    const int unit = blockIdx.x >> 1;
    const int units = gridDim.x >> 1;
    const int total_tiles = p.total_tiles;

    if (warp == 0) {
        if (lane == 0) {
            ptx::prefetch_tensormap(&tmap_w);
            for (int s = 0; s < p.stages; ++s) {
                ptx::mbar_init(full_bar(s), 1);
                ptx::mbar_init(empty_bar(s), 1);
            }
            for (int b = 0; b < 2; ++b) {
                ptx::mbar_init(tfull_bar(b), 1);
                ptx::mbar_init(tempty_bar(b), 8);    // one arrival per epilogue warp of both CTAs
            }
            ptx::fence_mbar_init();
        }
        __syncwarp();
    }
    if (warp == 1) {
        ptx::tmem_alloc_t<true>(tmem_slot, kTmemCols);
        ptx::tmem_relinquish_t<true>();
    }
    ptx::tc_fence_before();
    ptx::cluster_sync();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    ptx::pdl_launch_dependents();
    // W ahead of the wait (strict mode).  req_offsets[R] decides the decomposition, and it may only be read
    // after the wait - but a batch is usually dense, so the producer GUESSES the dense decomposition
    // (hint_C chunks, hint_S splits), requests the W boxes (the A operand) of its first `stages` pipeline
    // slots and asks L2 for the next `stages`.  The barrier of such a slot has the W bytes of both CTAs
    // pending but no arrival yet; the hidden boxes (whose height depends on the real chunk size) and the
    // arrival follow after the wait.  A wrong guess costs the boxes: they land, the issuer frees the
    // slots without a single MMA, and the pipeline starts over (flex_drop).
    int pre = 0;
    if (warp == 0 && p.wait_first && p.hint_C > 0 && unit < p.hint_C * p.hint_S) {
        const uint32_t full0 = ptx::mapa(full_bar(0), 0u);
        int tile = unit / p.hint_C, kb = 0;
        for (int slot = 0; slot < p.stages + p.prefetch_slots && tile < total_tiles; ++slot) {
            if (ptx::elect_one()) {
                const int a_row = tile * kFlexVocabTile + static_cast<int>(rank) * kTileM;
                if (slot < p.stages) {
                    if (rank == 0) ptx::mbar_expect_tx(full_bar(slot), 2u * kABytes);
                    ptx::tma_load_2d_pair(smem + static_cast<uint32_t>(slot) * p.stage_bytes, &tmap_w,
                                          full0 + 8u * slot, w_c0(p, kb), w_c1(p, kb, a_row), p.w_policy);
                } else {
                    ptx::tma_prefetch_2d(&tmap_w, w_c0(p, kb), w_c1(p, kb, a_row));
                }
            }
            __syncwarp();
            if (slot < p.stages) ++pre;
            if (++kb == p.k_blocks) { kb = 0; tile += p.hint_S; }
        }
    }
    LASER_TL(t.tl_slot, 1, 0);
    if (p.wait_first) ptx::pdl_wait();
    LASER_TL(t.tl_slot, 2, 0);
    uint32_t base = 0;
    const bool base_early = p.wait_first != 0;
    if (threadIdx.x == kTailThread0 && t.kind != 0 && base_early) base = ptx::ld_relaxed_gpu_u32(t.ctl + 1);
    int* off_c = reinterpret_cast<int*>(bars_gen + 256u);
    float* tau_c = reinterpret_cast<float*>(off_c + p.tail_cache + 1);
    const bool cached = t.kind == 1 && t.q.f.R <= p.tail_cache;
    if (cached && warp >= 2) {
        const FinalizeParams& f = t.q.f;
        for (int i = threadIdx.x - kTailThread0; i <= f.R; i += kEpilogueThreads) {
            off_c[i] = __ldg(f.req_offsets + i);
            if (i < f.R) tau_c[i] = tau_eval(__ldg(f.load + i), f.tau);
        }
    }

    const RunPlan rp = resolve_plan(p.pd);      // kind 3: uniform over the grid
    const int C = rp.m_items, S = rp.S, n_tok = rp.n_tok;
    const int work_items = C * S;               // item w: chunk w % C (fastest), split w / C
    const int half_tok = n_tok >> 1;            // token rows this CTA stages per chunk (B operand)
    const TailRole tr{p.grid_total, 0, static_cast<int>(gridDim.x)};
    // slots requested ahead of the wait (every warp can tell: the condition is the producer's) and whether
    // the guess they were requested under holds
    int pre_slots = 0;
    if (p.wait_first && p.hint_C > 0 && unit < p.hint_C * p.hint_S) {
        int tile = unit / p.hint_C, kb = 0;
        for (int slot = 0; slot < p.stages && tile < total_tiles; ++slot) {
            ++pre_slots;
            if (++kb == p.k_blocks) { kb = 0; tile += p.hint_S; }
        }
    }
    const bool flex_drop = pre_slots > 0 && (C != p.hint_C || S != p.hint_S);

    if (warp == 0) {
        // ===================================================================== TMA producer
        const CUtensorMap* tmap_h = &tm_hid.hid[(n_tok >> 4) - 1];
        if (lane == 0) ptx::prefetch_tensormap(tmap_h);
        const uint32_t txb2 = 2u * static_cast<uint32_t>(half_tok * 128);    // hidden bytes of both CTAs
        const uint32_t tx2 = 2u * kABytes + txb2;                            // W + hidden bytes of both CTAs
        const int k_blocks = p.k_blocks, stages = p.stages;
        const uint32_t full0 = ptx::mapa(full_bar(0), 0u);
        int stage = 0;
        uint32_t phase = 0;
        if (flex_drop) {
            // wrong guess: close the phases of the requested slots (the W bytes still land) and move on
            for (; pre > 0; --pre) {
                if (rank == 0 && ptx::elect_one()) ptx::mbar_arrive(full_bar(stage));
                __syncwarp();
                if (++stage == stages) { stage = 0; phase ^= 1u; }
            }
        }
        for (int w = unit; w < work_items; w += units) {
            const int c = w % C, sp = w / C;
            const int b_row = c * n_tok + static_cast<int>(rank) * half_tok;        // token rows
            for (int tile = sp; tile < total_tiles; tile += S) {
                const int a_row = tile * kFlexVocabTile + static_cast<int>(rank) * kTileM;   // vocabulary rows
                for (int kb = 0; kb < k_blocks; ++kb) {
                    const uint32_t sa = smem + static_cast<uint32_t>(stage) * p.stage_bytes;
                    const uint32_t fb = full0 + 8u * stage;
                    if (pre > 0) {
                        // the slot's W box went out ahead of the wait: its hidden box and the arrival
                        --pre;
                        if (ptx::elect_one()) {
                            if (rank == 0) ptx::mbar_arrive_expect_tx(full_bar(stage), txb2);
                            ptx::tma_load_2d_pair(sa + kABytes, tmap_h, fb, kb * kBlockK, b_row, ptx::kEvictLast);
                        }
                    } else {
                        ptx::mbar_wait(empty_bar(stage), phase ^ 1u);
                        if (ptx::elect_one()) {
                            if (rank == 0) ptx::mbar_arrive_expect_tx(full_bar(stage), tx2);
                            ptx::tma_load_2d_pair(sa, &tmap_w, fb, w_c0(p, kb), w_c1(p, kb, a_row), p.w_policy);
                            ptx::tma_load_2d_pair(sa + kABytes, tmap_h, fb, kb * kBlockK, b_row, ptx::kEvictLast);
                        }
                    }
                    __syncwarp();
                    if (++stage == stages) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================================================================== MMA issuer (leader CTA)
        if (rank == 0) {
            const uint32_t idesc = make_idesc_bf16(static_cast<uint32_t>(n_tok), 2 * kTileM);
            const uint64_t a_desc0 = make_smem_desc_sw128(smem);
            const uint64_t b_desc0 = make_smem_desc_sw128(smem + kABytes);
            const uint32_t stage_step = p.stage_bytes >> 4;
            const int k_blocks = p.k_blocks, stages = p.stages;
            int stage = 0;
            uint32_t phase = 0, acc = 0, desc_off = 0;
            if (flex_drop) {
                // boxes requested under a wrong guess: wait until they have landed, free the slots
                for (int i = 0; i < pre_slots; ++i) {
                    ptx::mbar_wait(full_bar(stage), phase);
                    if (ptx::elect_one()) ptx::umma_commit_t<true>(empty_bar(stage));
                    __syncwarp();
                    desc_off += stage_step;
                    if (++stage == stages) { stage = 0; phase ^= 1u; desc_off = 0; }
                }
            }
            for (int w = unit; w < work_items; w += units) {
                for (int tile = w / C; tile < total_tiles; tile += S, ++acc) {
                    const uint32_t buf = acc & 1u, aphase = (acc >> 1) & 1u;
                    ptx::mbar_wait_cluster(tempty_bar(buf), aphase ^ 1u);
                    ptx::tc_fence_after();
                    const uint32_t d_tmem = tmem_base + buf * kMaxTileN;
                    for (int kb = 0; kb < k_blocks; ++kb) {
                        ptx::mbar_wait(full_bar(stage), phase);
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
                            const uint64_t a_desc = a_desc0 + desc_off;
                            const uint64_t b_desc = b_desc0 + desc_off;
                            ptx::umma_bf16_t<true>(d_tmem, a_desc, b_desc, idesc, kb != 0);
                            ptx::umma_bf16_t<true>(d_tmem, a_desc + 2u, b_desc + 2u, idesc, 1u);
                            ptx::umma_bf16_t<true>(d_tmem, a_desc + 4u, b_desc + 4u, idesc, 1u);
                            ptx::umma_bf16_t<true>(d_tmem, a_desc + 6u, b_desc + 6u, idesc, 1u);
                            ptx::umma_commit_t<true>(empty_bar(stage));
                            if (kb == k_blocks - 1) ptx::umma_commit_t<true>(tfull_bar(buf));
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
        const int q = warp & 3;                  // TMEM lanes [32 q, 32 q + 32) = vocabulary rows of this warp
        const uint32_t lane_addr = static_cast<uint32_t>(q * 32) << 16;
        float* const xp = xpose + q * 1024;      // this warp's 32 x 32 transpose block
        const int nch = (n_tok + 31) >> 5;       // 32-token groups of a chunk (the last may hold 16)
        const int et = threadIdx.x - kTailThread0;   // 0..127
        uint32_t acc = 0;
        for (int w = unit; w < work_items; w += units) {
            const int c = w % C, sp = w / C;
            const int tok0 = c * n_tok;          // first token row of the chunk
            float m[8], s[8], lt[8];
            int a[8], tok[8];
#pragma unroll
            for (int ch = 0; ch < 8; ++ch) {
                m[ch] = -CUDART_INF_F; s[ch] = 0.f; lt[ch] = -CUDART_INF_F; a[ch] = -1; tok[ch] = -1;
            }
            if (p.token_ids != nullptr) {
#pragma unroll
                for (int ch = 0; ch < 8; ++ch) {
                    const int n = tok0 + 32 * ch + lane;
                    if (ch < nch && 32 * ch + lane < n_tok && n < p.n_alloc) {
                        const int tk = __ldg(p.token_ids + n) - p.v_offset;
                        tok[ch] = (tk >= 0 && tk < p.V) ? tk : -1;
                    }
                }
            }
            for (int tile = sp; tile < total_tiles; tile += S, ++acc) {
                const uint32_t buf = acc & 1u, aphase = (acc >> 1) & 1u;
                ptx::mbar_wait(tfull_bar(buf), aphase);
                ptx::tc_fence_after();
                const uint32_t taddr = tmem_base + lane_addr + buf * kMaxTileN;
                const int v0 = tile * kFlexVocabTile + static_cast<int>(rank) * kTileM + q * 32;
                const bool any_v = v0 < p.V;     // rows past the end of W (TMA zero fill): nothing to fold
#pragma unroll
                for (int ch = 0; ch < 8; ++ch) {
                    if (ch < nch) {
                        uint32_t r[32];
                        ptx::tmem_ld_x32(taddr + 32 * ch, r);
                        ptx::tmem_wait_ld();
                        if (ch == nch - 1) {
                            // every TMEM read of this warp has completed: release the accumulator
                            ptx::tc_fence_before();
                            __syncwarp();
                            if (lane == 0) ptx::mbar_arrive_cluster(ptx::mapa(tempty_bar(buf), 0u));
                        }
                        if (any_v) {
                            // r[j] = logit(vocabulary row v0 + lane, token 32 ch + j)  ->  y[k] = logit(v0 + k, token 32 ch + lane)
                            __syncwarp();        // the previous block's reads are done
#pragma unroll
                            for (int j = 0; j < 32; ++j)
                                xp[j * 32 + 4 * ((lane >> 2) ^ (j & 7)) + (lane & 3)] = __uint_as_float(r[j]);
                            __syncwarp();
                            uint32_t y[32];
#pragma unroll
                            for (int k = 0; k < 8; ++k) {
                                const uint4 v = *reinterpret_cast<const uint4*>(xp + lane * 32 + 4 * (k ^ (lane & 7)));
                                y[4 * k] = v.x; y[4 * k + 1] = v.y; y[4 * k + 2] = v.z; y[4 * k + 3] = v.w;
                            }
                            fold_columns<32>(y, v0, p.V, m[ch], a[ch], s[ch], tok[ch], lt[ch]);
                        }
                    }
                }
            }
            // ---- the four warps hold four vocabulary quarters of every token: merge through shared memory.
            // Warp q's records of tokens [0, 256) fill exactly its own 4 KB block.
            __syncwarp();
            float4* const rec = reinterpret_cast<float4*>(xpose);
#pragma unroll
            for (int ch = 0; ch < 8; ++ch)
                if (ch < nch) rec[q * 256 + 32 * ch + lane] = make_float4(m[ch], s[ch], __int_as_float(a[ch]), lt[ch]);
            group_sync<3, kEpilogueThreads>();
            if (p.role != 1) ptx::pdl_wait();    // overlap mode: the previous call's tail may still read the workspace
            for (int tk = et; tk < n_tok; tk += kEpilogueThreads) {
                const int n = tok0 + tk;
                float4 v[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) v[i] = rec[i * 256 + tk];
                const float M = fmaxf(fmaxf(v[0].x, v[1].x), fmaxf(v[2].x, v[3].x));
                float sum = 0.f, l = -CUDART_INF_F;
                int am = 0x7fffffff;
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const float sc = (v[i].x == M) ? 1.f : ptx::ex2_approx((v[i].x - M) * kLog2e);
                    sum += v[i].y * sc;
                    if (v[i].x == M) am = min(am, __float_as_int(v[i].z));   // equal maxima: the lower index
                    l = fmaxf(l, v[i].w);
                }
                if (n < p.n_alloc)
                    p.ws[static_cast<int64_t>(n) * (2 * S) + 2 * sp + static_cast<int>(rank)] =
                        make_float4(M, sum, __int_as_float(am), l);
            }
            group_sync<3, kEpilogueThreads>();   // the blocks are transpose scratch again
        }
        LASER_TL(t.tl_slot, 3, kTailThread0);
        ptx::tc_fence_before();
        ptx::cluster_arrive();
        if (t.kind != 0) {
            float* scratch = reinterpret_cast<float*>(bars_gen + 192u);
            fused_tail(p, t, rp, tr, base, base_early, cached, off_c, tau_c, scratch);
        }
    }

    // ------------------------------------------------------------------------- teardown
    __syncwarp();
    LASER_TL(t.tl_slot, 7, 0);
    ptx::pdl_wait();
    if (warp >= 2) {
        ptx::cluster_wait();
        return;
    }
    ptx::tc_fence_before();
    ptx::cluster_sync();
    if (warp == 1) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc_t<true>(tmem_base, kTmemCols);
    }
}

}  // namespace laser
