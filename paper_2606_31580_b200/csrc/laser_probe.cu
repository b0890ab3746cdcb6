// laser_probe.cu — host side of the C ABI declared in include/laser_probe.h: argument validation,
// launch planning, TMA descriptor encoding (driver entry point fetched through the runtime, no
// -lcuda), probe handles (plan + encoded descriptors + control slot cached once) and the kernel
// launches.  No per-call device allocation, no host<->device synchronisation (except in the explicit
// *_host entry points), no fallback path.
#include "../../include/laser_probe.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <deque>
#include <mutex>
#include <string>
#include <vector>

#include "probe_kernels.cuh"
#include "flex_kernel.cuh"

namespace {

using namespace laser;

thread_local std::string g_last_error;
std::atomic<uint64_t> g_launches{0};

// Optional per-kernel timing (bench / profiling only): when enabled on this thread, every call
// records events before the fused kernel, after it and after the finalize kernel (if there is one).
constexpr int kProfRing = 512;
struct ProfState {
    bool on = false;
    int calls = 0;
    cudaEvent_t ev[kProfRing][3] = {};
    bool created = false;
};
thread_local ProfState g_prof;

constexpr int kDefaultSMs = 148;             // B200
constexpr int kMaxDynSmem = 227 * 1024;      // per-CTA opt-in limit on sm_100
constexpr int kSmemSlack = 1024 + 256;       // alignment slack + barrier block
constexpr int kCtlSlots = 4096;              // control slots per device
constexpr int kCtlWords = 4;                 // words per slot (see TailParams)

int set_cuda_error(const char* what, cudaError_t e) {
    g_last_error = std::string(what) + ": " + cudaGetErrorString(e);
    return LASER_E_CUDA;
}

// ---------------------------------------------------------------------------------------- device
struct DeviceInfo {
    bool queried = false, ok = false;
    int sms = kDefaultSMs, cc_major = 0, cc_minor = 0;
    bool attr_set = false;
    // control block: kCtlSlots x kCtlWords counters (see TailParams)
    uint32_t* ctl_base = nullptr;
    bool ctl_failed = false;
    std::deque<int> ctl_free;
};
std::mutex g_mu;
DeviceInfo g_dev[64];

// Returns the cached info of the current device; cuda_ok = false if no device can be queried.
DeviceInfo* current_device(bool* cuda_ok) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) {
        (void)cudaGetLastError();
        *cuda_ok = false;
        return nullptr;
    }
    DeviceInfo& d = g_dev[dev];
    if (!d.queried) {
        std::lock_guard<std::mutex> lk(g_mu);
        if (!d.queried) {
            d.ok = cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess &&
                   cudaDeviceGetAttribute(&d.cc_major, cudaDevAttrComputeCapabilityMajor, dev) == cudaSuccess &&
                   cudaDeviceGetAttribute(&d.cc_minor, cudaDevAttrComputeCapabilityMinor, dev) == cudaSuccess;
            if (!d.ok) (void)cudaGetLastError();
            d.queried = true;
        }
    }
    *cuda_ok = d.ok;
    return &d;
}

// A control slot of the current device, or nullptr (none left / allocation failed / `stream` is
// being captured before the block exists: cudaMalloc is not allowed under capture).
uint32_t* acquire_ctl(DeviceInfo* di, cudaStream_t stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!di->ctl_base) {
        if (di->ctl_failed) return nullptr;
        // The caller's stream may be under capture (nothing can be allocated then).  The legacy stream
        // (nullptr: laser_probe_handle_create, or a caller on the default stream) cannot be captured, and
        // merely querying it while ANOTHER thread captures in global mode would invalidate that capture.
        if (stream != nullptr) {
            cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
            if (cudaStreamIsCapturing(stream, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) {
                (void)cudaGetLastError();
                return nullptr;   // retried by the next call outside a capture
            }
        }
        // One-time allocation.  This thread's capture mode is relaxed for its duration, so that the calls
        // below do not break a capture some other thread has open; the zeroes are on the device before any
        // kernel of any stream (torch's streams do not synchronise with the legacy stream) can read them.
        cudaStreamCaptureMode cmode = cudaStreamCaptureModeRelaxed;
        const bool exchanged = cudaThreadExchangeStreamCaptureMode(&cmode) == cudaSuccess;
        void* p = nullptr;
        bool ok = cudaMalloc(&p, sizeof(uint32_t) * kCtlWords * kCtlSlots) == cudaSuccess;
        if (ok) {
            cudaStream_t zs = nullptr;
            ok = cudaStreamCreateWithFlags(&zs, cudaStreamNonBlocking) == cudaSuccess;
            if (ok) {
                ok = cudaMemsetAsync(p, 0, sizeof(uint32_t) * kCtlWords * kCtlSlots, zs) == cudaSuccess &&
                     cudaStreamSynchronize(zs) == cudaSuccess;
                (void)cudaStreamDestroy(zs);
            }
            if (!ok) (void)cudaFree(p);
        }
        if (exchanged) (void)cudaThreadExchangeStreamCaptureMode(&cmode);
        if (!ok) {
            (void)cudaGetLastError();
            di->ctl_failed = true;
            return nullptr;
        }
        di->ctl_base = static_cast<uint32_t*>(p);
        for (int i = 0; i < kCtlSlots; ++i) di->ctl_free.push_back(i);
    }
    if (di->ctl_free.empty()) return nullptr;
    const int slot = di->ctl_free.front();
    di->ctl_free.pop_front();
    return di->ctl_base + kCtlWords * slot;
}
void release_ctl(DeviceInfo* di, uint32_t* ctl) {
    if (!ctl || !di) return;
    std::lock_guard<std::mutex> lk(g_mu);
    if (di->ctl_base) di->ctl_free.push_back(static_cast<int>((ctl - di->ctl_base) / kCtlWords));  // FIFO: reused last
}

// ---------------------------------------------------------------------------------------- plan
int ceil_div(int a, int b) { return (a + b - 1) / b; }
int round_up(int a, int b) { return ceil_div(a, b) * b; }
int gcd_i(int a, int b) { while (b) { int t = a % b; a = b; b = t; } return a; }

bool dims_valid(const laser_probe_dims* d) {
    return d && d->d > 0 && d->V > 0 && d->N >= 0 && d->R >= 0 && (d->d % 8) == 0;
}

// Choose (splits, tiles_per_split, tile_n) for one kernel variant.  A "unit" is what executes a work
// item: a CTA (single mode, 128 token rows) or a CTA pair (pair mode, 256 token rows).  The
// vocabulary is cut into splits of T*BN rows, BN a multiple of `bn_step` and <= 256.  m_tiles*splits
// should fill the units in whole rounds; among such choices minimise the busiest unit's work, counted
// in W rows plus a charge per tile for re-streaming the hidden rows from L2.
double plan_variant(const laser_probe_dims& dm, int units, int tile_m, int bn_step, int* oS, int* oT,
                    int* oBN) {
    const int m_tiles = dm.N > 0 ? ceil_div(dm.N, tile_m) : 1;
    const int s_unit = units / gcd_i(units, m_tiles);
    const double kTileCharge = 32.0;  // W-row equivalents per tile (hidden re-stream, pipeline bubble)
    double best = 1e300;
    int bS = 1, bT = 1, bBN = bn_step;
    for (int k = 1; k <= 4; ++k) {
        const int s_try = s_unit * k;
        const int L = ceil_div(dm.V, s_try);
        const int t_min = ceil_div(L, kMaxTileN);
        for (int T = t_min; T <= t_min + 3; ++T) {
            const int BN = round_up(ceil_div(L, T), bn_step);
            if (BN > kMaxTileN) continue;
            const int S = ceil_div(dm.V, T * BN);
            const long items = static_cast<long>(m_tiles) * S;
            const long rounds = (items + units - 1) / units;
            const double cost = static_cast<double>(rounds) * T * (BN + kTileCharge);
            if (cost < best - 1e-9) { best = cost; bS = S; bT = T; bBN = BN; }
        }
    }
    *oS = bS; *oT = bT; *oBN = bBN;
    return best;
}

// Plan of one kernel variant: CTA pairs (tcgen05 cta_group::2, M = 256; each W tile enters a pair's
// shared memory once instead of once per 128-row token tile and one issuing thread feeds two SMs'
// tensor cores: measured +10..17 % for N >= 256) or single CTAs (M = 128).  bn_force > 0 fixes tile_n.
void make_variant_plan(const laser_probe_dims& dm, int num_sms, bool pair, int bn_force, laser_probe_plan* pl) {
    const int tile_m = pair ? 2 * kTileM : kTileM;
    const int units = pair ? (num_sms / 2 > 0 ? num_sms / 2 : 1) : num_sms;
    int S, T, BN;
    plan_variant(dm, units, tile_m, pair ? 32 : 16, &S, &T, &BN);   // fixes the tile height BN
    if (bn_force > 0) BN = bn_force;
    memset(pl, 0, sizeof *pl);
    pl->num_sms = num_sms;
    pl->m_tiles = dm.N > 0 ? ceil_div(dm.N, tile_m) : 1;
    // The deal of tiles to units comes from the function the kernels also use: with padding rows in
    // the batch they re-plan on the device for the token items that hold rows (same BN).
    const int total_tiles = ceil_div(dm.V, BN);
    const SplitPlan sp = plan_splits(total_tiles, pl->m_tiles, units);
    S = sp.splits; T = sp.T;
    // packed records: the most any item count m <= m_tiles can write
    long ws_records = static_cast<long>(pl->m_tiles) * tile_m * S;
    for (int m = 1; m < pl->m_tiles; ++m) {
        const long rec = static_cast<long>(m) * tile_m * plan_splits(total_tiles, m, units).splits;
        if (rec > ws_records) ws_records = rec;
    }
    pl->ws_records = static_cast<int32_t>(ws_records);
    pl->splits = S;
    pl->tiles_per_split = T;
    pl->tile_n = BN;
    pl->k_blocks = ceil_div(dm.d, kBlockK);
    const int stage_bytes = kABytes + (pair ? BN / 2 : BN) * 128;
    int stages = (kMaxDynSmem - kSmemSlack) / stage_bytes;
    if (stages > kMaxStages) stages = kMaxStages;
    pl->stages = stages;
    pl->work_items = pl->m_tiles * S;
    const int busy = pl->work_items < units ? pl->work_items : units;
    pl->grid = pair ? 2 * busy : busy;
    // what the pipeline leaves over holds the tail's {offset, threshold} cache: 8 bytes per request
    const int spare = kMaxDynSmem - (stages * stage_bytes + kSmemSlack);
    int cache = spare / 8 - 1;
    if (cache > kTailCache) cache = kTailCache;
    if (cache < 0) cache = 0;
    pl->tail_cache = cache;
    pl->smem_bytes = stages * stage_bytes + kSmemSlack + (cache > 0 ? 8 * (cache + 1) : 0);
    pl->kernel_launches = 1;
    pl->tile_m = tile_m;
    pl->cta_pair = pair ? 1 : 0;
}

// ---- mixed schedule: the host plans every count of 128-row tiles that may hold rows
// Cost model (B200, measured): a pair CTA spends 2*128*bn*d flop / 10 TFLOP/s on its
// half of a 256-row item's tile; a single CTA needs 1.2x that for a 128-row tile (it stages a whole W
// tile instead of half of one: 1.31x at boost clocks, 1.09x under the power cap); every kernel that
// takes part streams W from HBM once (6.4 TB/s), and the second kernel of a call starts a few
// microseconds behind the first.
struct MixedChoice { int sched, u_tail, S_pair, S_tail, k_pair, j_single; double time; };
MixedChoice plan_mixed_host(int m128, int V, int d, int bn_pair, int bn_tail, int sms) {
    const int tiles_pair = ceil_div(V, bn_pair), tiles_tail = ceil_div(V, bn_tail);
    const double t_p = 2.0 * kTileM * bn_pair * d / 10.0e12, t_s = 1.2 * 2.0 * kTileM * bn_tail * d / 10.0e12;
    const double hbm_pass = 2.0 * V * d / 6.4e12;
    const int pairs = sms / 2 > 0 ? sms / 2 : 1;
    auto part = [](int tiles, int items, int units, double t_tile, int* S) {
        const SplitPlan sp = plan_splits(tiles, items, units);
        *S = sp.splits;
        const long rounds = (static_cast<long>(items) * sp.splits + units - 1) / units;
        return static_cast<double>(rounds) * sp.T * t_tile;
    };
    MixedChoice best{0, 0, 1, 1, 0, 0, 1e300};
    {   // pair items only (an odd count pads half an item)
        MixedChoice c{0, 0, 1, 1, (m128 + 1) / 2, 0, 0.0};
        c.time = std::max(part(tiles_pair, c.k_pair, pairs, t_p, &c.S_pair), hbm_pass);
        best = c;
    }
    {   // single-CTA tiles only
        MixedChoice c{2, sms > 255 ? 255 : sms, 1, 1, 0, m128, 0.0};
        c.time = std::max(part(tiles_tail, m128, c.u_tail, t_s, &c.S_tail), hbm_pass);
        if (c.time < best.time) best = c;
    }
    if ((m128 & 1) && m128 >= 3) {   // pair items + the odd tile on single CTAs, side by side
        for (int ut = 2; ut <= sms - 2 && ut <= 254; ut += 2) {   // whole TPCs: see launch_fused
            MixedChoice c{1, ut, 1, 1, m128 / 2, 1, 0.0};
            const double ta = part(tiles_pair, c.k_pair, (sms - ut) / 2, t_p, &c.S_pair);
            const double tb = part(tiles_tail, 1, ut, t_s, &c.S_tail);
            // two W passes at once do not reach the single-stream rate (5.5 instead of 6.4 TB/s)
            c.time = std::max(std::max(ta + 4e-6, tb), 2.0 * hbm_pass * (6.4 / 5.5)) + 2e-6;
            if (c.time < best.time) best = c;
        }
    }
    return best;
}

// ---- flex kernel (flex_kernel.cuh): C chunks of n_tok token rows (multiple of 16, <= 256) x S vocabulary
// splits of 256-row tiles on the CTA pairs.  Cost of a (tile, chunk): the MMAs take time in proportion to
// n_tok; staging the 256 W rows, the pipeline bubble between tiles and the epilogue's fixed part are charged
// as kFlexTileCharge token rows.  Among the chunk counts that cover the rows the cheapest busiest pair wins.
struct FlexChoice { int C, n_tok, S, T, rounds; double cost; long busiest; };
// measured at the C2 shape: a (tile, chunk) takes 3.1 us + 0.028 us per token row
double flex_tile_charge() { return 110.0; }
FlexChoice plan_flex_host(int n_valid, int V, int sms) {
    const int pairs = sms / 2 > 0 ? sms / 2 : 1;
    const int tiles = ceil_div(V, kFlexVocabTile);
    FlexChoice best{0, 16, 1, tiles, 0, 1e300, 0};
    if (n_valid <= 0) { best.cost = 0.0; return best; }
    const int c_min = ceil_div(n_valid, kFlexMaxTok);
    for (int C = c_min; C <= c_min + 3 && C <= 31; ++C) {
        const int n_tok = round_up(ceil_div(n_valid, C), 16);
        if (n_tok > kFlexMaxTok) continue;
        // splits in multiples of the smallest count that fills the pairs in whole rounds: every pair
        // streams W (the tiles of a split are dealt round-robin, so splits differ by at most one tile)
        const int s_unit = pairs / gcd_i(pairs, C);
        for (int k = 1; k <= 4; ++k) {
            int S = s_unit * k;
            if (S > tiles) { if (k > 1) break; S = tiles; }     // tiny vocabularies: a tile per split
            const int T = ceil_div(tiles, S);
            const long rounds = (static_cast<long>(C) * S + pairs - 1) / pairs;
            // the busiest pair, exactly: pair u takes items u, u + pairs, ...; item w is split w / C
            long busiest = 0;
            for (int u = 0; u < pairs && u < C * S; ++u) {
                long tl = 0;
                for (int w = u; w < C * S; w += pairs) {
                    const int sp = w / C;
                    tl += sp < tiles ? (tiles - sp + S - 1) / S : 0;
                }
                if (tl > busiest) busiest = tl;
            }
            const double cost = static_cast<double>(busiest) * (n_tok + flex_tile_charge()) + 8.0 * rounds;
            if (cost < best.cost - 1e-9) best = FlexChoice{C, n_tok, S, T, static_cast<int>(rounds), cost, busiest};
        }
    }
    return best;
}

// Plan of the flex kernel for dims (N <= kFlexMaxRows) and its table: entry [g - 1] for g 16-row groups.
void make_flex_plan(const laser_probe_dims& dm, int num_sms, laser_probe_plan* pl, uint32_t* tab) {
    memset(pl, 0, sizeof *pl);
    const int groups = ceil_div(dm.N, 16);
    int max_tok = 16;
    long ws_records = 1;
    FlexChoice dense{0, 16, 1, 1, 0, 0.0, 0};
    for (int g = 1; g <= kMixedTabMax; ++g) {
        const int gg = g <= groups ? g : (groups > 0 ? groups : 1);
        const int n_valid = gg * 16 < dm.N ? gg * 16 : (dm.N > 0 ? dm.N : 16);
        const FlexChoice c = plan_flex_host(n_valid, dm.V, num_sms);
        if (tab) tab[g - 1] = flex_pack(c.C, c.n_tok, c.S);
        if (g > groups && groups > 0) continue;
        if (c.n_tok > max_tok) max_tok = c.n_tok;
        long rows = static_cast<long>(c.C) * c.n_tok;
        if (rows > dm.N) rows = dm.N;
        const long rec = rows * 2L * c.S;
        if (rec > ws_records) ws_records = rec;
        if (g == groups) dense = c;
    }
    pl->num_sms = num_sms;
    pl->m_tiles = dense.C > 0 ? dense.C : 1;
    pl->splits = dense.S;
    pl->tiles_per_split = dense.T;
    pl->tile_n = kFlexVocabTile;
    pl->k_blocks = ceil_div(dm.d, kBlockK);
    const int stage_bytes = kABytes + (max_tok / 2) * 128;
    int stages = (kMaxDynSmem - kSmemSlack - kFlexXposeBytes) / stage_bytes;
    if (stages > kMaxStages) stages = kMaxStages;
    pl->stages = stages;
    pl->work_items = pl->m_tiles * pl->splits;
    pl->grid = 2 * (num_sms / 2 > 0 ? num_sms / 2 : 1);
    const int spare = kMaxDynSmem - (stages * stage_bytes + kSmemSlack + kFlexXposeBytes);
    int cache = spare / 8 - 1;
    if (cache > kTailCache) cache = kTailCache;
    if (cache < 0) cache = 0;
    pl->tail_cache = cache;
    pl->smem_bytes = stages * stage_bytes + kSmemSlack + kFlexXposeBytes + (cache > 0 ? 8 * (cache + 1) : 0);
    pl->kernel_launches = 1;
    pl->tile_m = dense.n_tok;
    pl->cta_pair = 1;
    pl->ws_records = static_cast<int32_t>(ws_records);
    pl->flex = 1;
    pl->flex_n_tok = dense.n_tok;
    pl->flex_max_tok = max_tok;
}

// AUTO: one single-CTA kernel for N <= 128 rows; above that the mixed schedule (probe_kernels.cuh):
// 256-row items on CTA pairs and / or 128-row tiles on single CTAs - which, is looked up on the device
// from the number of 128-row tiles that hold rows (req_offsets[R]), so a padded batch pays for the
// rows it holds.  *tail_pl (mixed only) is the plan of the single-CTA kernel.
// SINGLE / PAIR force one variant (an odd tile count then costs the pair kernel a padding tile).
void make_plan(const laser_probe_dims& dm, int num_sms, int mode, laser_probe_plan* pl, laser_probe_plan* tail_pl) {
    const int t128 = ceil_div(dm.N, kTileM);
    // AUTO takes the flex kernel for 129..1024 allocated rows except exactly 256 (measured at the C2 / C3 /
    // C4 shapes: it wins wherever the rows do not fill 256-row items - N = 320: 130 vs 151 us,
    // C4's 590 of 1024 rows: 456 vs 508 us - and ties at 512 / 768 / 1024; a dense 256-row batch is the
    // one case where its fixed 256-row vocabulary tiles quantise worse than the pair kernel's).
    bool auto_flex = mode == LASER_MODE_AUTO && dm.N > kTileM && dm.N <= 1024 && dm.N != 2 * kTileM;
    // Narrow hidden sizes: a tile's MMAs shrink with d, its epilogue does not, and the flex epilogue is ~30 %
    // heavier (the 32 x 32 transposes).  Measured at V = 151936 (flex vs mixed, strict step): d = 1024 N = 320
    // 96 vs 103 us but N = 512 132 vs 121; d = 512 N = 320 72 vs 59.  Below d = 1280 AUTO takes the flex
    // kernel only where the mixed schedule pays for padding tiles (N <= 384), below d = 768 not at all.
    const int kb_d = ceil_div(dm.d, kBlockK);
    if (auto_flex && (kb_d < 12 || (kb_d < 20 && dm.N > 384))) auto_flex = false;
    if (auto_flex) {
        // The flex kernel's vocabulary tiles are 256 rows whatever V is: with few tiles per pair (a small
        // vocabulary, a vocabulary shard) whole-tile quantisation can leave the busiest pair far above the
        // average - V = 18992 rows are 75 tiles for 74 pairs, one pair takes two.  The pair kernel picks its
        // tile height to fit, so AUTO keeps the former schedule when the busiest pair would carry more than
        // 15 % above an even share (C2's shape: 9 tiles against 8.03, 12 %).
        const FlexChoice c = plan_flex_host(dm.N, dm.V, num_sms);
        const int pairs = num_sms / 2 > 0 ? num_sms / 2 : 1;
        const double even = static_cast<double>(ceil_div(dm.V, kFlexVocabTile)) * c.C / pairs;
        if (static_cast<double>(c.busiest) > 1.15 * (even > 1.0 ? even : 1.0)) auto_flex = false;
    }
    if ((mode == LASER_MODE_FLEX && dm.N > 0 && dm.N <= kFlexMaxRows) || auto_flex) {
        make_flex_plan(dm, num_sms, pl, nullptr);
        return;
    }
    if (mode == LASER_MODE_FLEX || mode == LASER_MODE_MIXED) mode = LASER_MODE_AUTO;     // the schedule AUTO had before
    if (mode == LASER_MODE_SINGLE || (mode == LASER_MODE_AUTO && t128 <= 1)) {
        make_variant_plan(dm, num_sms, false, 0, pl);
        return;
    }
    make_variant_plan(dm, num_sms, true, 0, pl);
    if (mode == LASER_MODE_PAIR) return;
    // 129..256 rows: one 256-row pair item whatever req_offsets[R] says - a static plan (one launch, W
    // requested ahead of the wait, tail in the kernel).  With <= 128 valid rows half the item is padding,
    // which costs little: that case is bound by the W stream.
    if (t128 == 2) return;
    // ---- mixed
    laser_probe_dims d1 = dm;
    d1.N = kTileM;
    // the single-CTA kernel keeps the tile height that balances one 128-row tile over all SMs (the
    // case where it works alone); on a fraction of the SMs it has many tiles per CTA anyway
    laser_probe_plan tp;
    make_variant_plan(d1, num_sms, false, 0, &tp);
    tp.grid = num_sms;           // every SM may be needed (single-CTA tiles only)
    pl->grid = 2 * (num_sms / 2 > 0 ? num_sms / 2 : 1);
    pl->mixed = 1;
    pl->tail_tile_n = tp.tile_n;
    pl->tail_stages = tp.stages;
    pl->tail_smem_bytes = tp.smem_bytes;
    pl->tail_grid = tp.grid;
    pl->kernel_launches = 2;     // single-CTA kernel, pair kernel (+ finalize kernel: LASER_TAIL_SEPARATE)
    long ws_records = 1;
    for (int m128 = 1; m128 <= t128; ++m128) {
        long rec;
        if (m128 < kMixedTabMax) {
            const MixedChoice c = plan_mixed_host(m128, dm.V, dm.d, pl->tile_n, tp.tile_n, num_sms);
            rec = 2L * kTileM * c.k_pair * c.S_pair + static_cast<long>(kTileM) * c.j_single * c.S_tail;
        } else {
            const int k = (m128 + 1) / 2, up = num_sms / 2 > 0 ? num_sms / 2 : 1;
            rec = 2L * kTileM * k * plan_splits(ceil_div(dm.V, pl->tile_n), k, up).splits;
        }
        if (rec > ws_records) ws_records = rec;
    }
    pl->ws_records = static_cast<int32_t>(ws_records);
    if (tail_pl) *tail_pl = tp;
}

// The table of PlanDesc (kind 2): one packed plan per count of 128-row tiles.
void fill_mixed_table(const laser_probe_dims& dm, const laser_probe_plan& pl, int num_sms, uint32_t* tab) {
    const int t128 = ceil_div(dm.N, kTileM);
    tab[0] = mixed_pack(0, 0, 1, 1);
    for (int m128 = 1; m128 < kMixedTabMax; ++m128) {
        if (m128 > t128) { tab[m128] = tab[t128 < kMixedTabMax ? t128 : kMixedTabMax - 1]; continue; }
        const MixedChoice c = plan_mixed_host(m128, dm.V, dm.d, pl.tile_n, pl.tail_tile_n, num_sms);
        tab[m128] = mixed_pack(c.sched, c.u_tail, c.S_pair, c.S_tail);
    }
}

size_t workspace_bytes_for(const laser_probe_plan& pl) {
    size_t b = static_cast<size_t>(16) * static_cast<size_t>(pl.ws_records);
    return b < 16 ? 16 : b;
}

// ---------------------------------------------------------------------------------------- TMA maps
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
std::atomic<EncodeTiledFn> g_encode{nullptr};

// bf16 [rows, cols] row-major; box = 64 columns (128 B, the swizzle span) x box_rows rows.
int encode_tensor_map(const void* ptr, int rows, int cols, int box_rows, CUtensorMap* out) {
    EncodeTiledFn enc = g_encode.load(std::memory_order_acquire);
    if (!enc) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) {
            (void)cudaGetLastError();
            g_last_error = "cudaGetDriverEntryPoint(cuTensorMapEncodeTiled) failed";
            return LASER_E_CUDA;
        }
        enc = reinterpret_cast<EncodeTiledFn>(fn);
        g_encode.store(enc, std::memory_order_release);
    }
    const cuuint64_t gdim[2] = {static_cast<cuuint64_t>(cols), static_cast<cuuint64_t>(rows)};
    const cuuint64_t gstride[1] = {static_cast<cuuint64_t>(cols) * 2};
    const cuuint32_t box[2] = {static_cast<cuuint32_t>(kBlockK), static_cast<cuuint32_t>(box_rows)};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), gdim,
                     gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        char buf[160];
        snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed (CUresult %d) rows=%d cols=%d box_rows=%d",
                 static_cast<int>(r), rows, cols, box_rows);
        g_last_error = buf;
        return LASER_E_CUDA;
    }
    return LASER_OK;
}

bool params_valid(const laser_tau_params* t) {
    return std::isfinite(t->lambda_base) && std::isfinite(t->beta) && std::isfinite(t->gamma) &&
           std::isfinite(t->l_target) && std::isfinite(t->lambda_min) && std::isfinite(t->lambda_max) &&
           t->l_target > 0.f && t->lambda_min <= t->lambda_max;
}

TauParamsDev to_dev(const laser_tau_params* t) {
    return TauParamsDev{t->lambda_base, t->beta, t->gamma, t->l_target, t->lambda_min, t->lambda_max};
}

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Staging {
    size_t hidden, offsets, load, conf, argmax, exit_, total;
};
Staging staging_layout(const laser_probe_dims& d) {
    Staging s;
    size_t o = 0;
    s.hidden = o;  o = align_up(o + static_cast<size_t>(d.N) * d.d * 2, 256);
    s.offsets = o; o = align_up(o + static_cast<size_t>(d.R + 1) * 4, 256);
    s.load = o;    o = align_up(o + static_cast<size_t>(d.R) * 4, 256);
    s.conf = o;    o = align_up(o + static_cast<size_t>(d.R) * 4, 256);
    s.argmax = o;  o = align_up(o + static_cast<size_t>(d.N) * 4, 256);
    s.exit_ = o;   o = align_up(o + static_cast<size_t>(d.R), 256);
    s.total = o < 256 ? 256 : o;
    return s;
}

const laser_probe_options kDefaultOptions{LASER_AGG_MEAN, LASER_PROB_MAX, nullptr, LASER_MODE_AUTO, 0,
                                          LASER_TAIL_AUTO, 0, 0};

// Everything but token_ids (checked per call: it may be supplied at run time).
int options_valid(const laser_probe_options& o) {
    if (o.aggregate_mode < LASER_AGG_MEAN || o.aggregate_mode > LASER_AGG_MIN) return LASER_E_MODE;
    if (o.prob_mode < LASER_PROB_MAX || o.prob_mode > LASER_PROB_TOKEN) return LASER_E_MODE;
    if (o.kernel_mode < LASER_MODE_AUTO || o.kernel_mode > LASER_MODE_MIXED) return LASER_E_MODE;
    if (o.tail < LASER_TAIL_AUTO || o.tail > LASER_TAIL_SEPARATE) return LASER_E_MODE;
    if (o.overlap != 0 && o.overlap != 1) return LASER_E_MODE;
    if (o.w_layout != LASER_W_ROWMAJOR && o.w_layout != LASER_W_KBLOCKED) return LASER_E_MODE;
    if (o.w_ordered != 0 && o.w_ordered != 1) return LASER_E_MODE;
    return LASER_OK;
}

// sm_100 only, no fallback.
int require_b200(DeviceInfo** out) {
    bool ok = false;
    DeviceInfo* di = current_device(&ok);
    if (!ok || !di) { g_last_error = "no usable CUDA device"; return LASER_E_CUDA; }
    if (di->cc_major != 10 || di->cc_minor != 0) return LASER_E_ARCH;
    *out = di;
    return LASER_OK;
}

// W boxes a producer asks L2 for ahead of griddepcontrol.wait, behind the `stages` boxes it requests into
// shared memory.  Measured at C2 (strict loop): 0 / 1 / 2 / 3 / 4 x stages = 77.2 / 77.5 / 77.9 / 76.5 / 78.1 us
// (row-major W; noise): one ring's worth is kept.
int prefetch_slots_for(int stages) { return stages; }

int units_for(const DeviceInfo* di, bool pair) { return pair ? (di->sms / 2 > 0 ? di->sms / 2 : 1) : di->sms; }

}  // namespace

// ============================================================================================ handle
// Everything about a probe of fixed dims + options that does not change from call to call: the
// launch plan, the encoded TMA descriptors of the (few) hidden / W buffers it is called with, the
// device-mapped addresses of pinned host buffers, and the control slot of the fused tail.  A call
// through a handle takes no lock and does no hashing.  Not thread-safe: one thread at a time.
struct laser_probe_handle_s {
    laser_probe_dims dims;
    laser_probe_options opt;
    laser_probe_plan plan;
    laser_probe_plan tail_plan;     // mixed schedule: the single-CTA kernel
    uint32_t mixed_tab[kMixedTabMax] = {};
    DeviceInfo* di = nullptr;
    uint32_t* ctl = nullptr;
    bool debug = false;
    struct MapEntry { const void* ptr = nullptr; int box_rows = 0; CUtensorMap map; };
    MapEntry hid[2], w[4];
    int hid_rr = 0, w_rr = 0;
    // flex kernel: one hidden map per chunk height (box of 8, 16, ..., 128 token rows), per hidden buffer
    struct FlexEntry { const void* ptr = nullptr; FlexMaps maps; };
    FlexEntry flex_hid[2];
    int flex_rr = 0;
    struct HostMap { const void* h = nullptr; void* d = nullptr; };
    HostMap hm[8];
    int hm_rr = 0;
    // set by run_host around its probe call: `hidden` is produced on the stream just ahead (the staging
    // kernel or the H2D copy), so the fused kernel must not read it before that work has completed,
    // whatever opt.overlap says
    bool strict_inputs = false;
};

namespace {

typedef laser_probe_handle_s Handle;

int handle_tensor_map(Handle::MapEntry* tab, int n, int* rr, const void* ptr, int rows, int cols,
                      int box_rows, const CUtensorMap** out) {
    for (int i = 0; i < n; ++i)
        if (tab[i].ptr == ptr && tab[i].box_rows == box_rows) { *out = &tab[i].map; return LASER_OK; }
    Handle::MapEntry& e = tab[*rr];
    *rr = (*rr + 1) % n;
    e.ptr = nullptr;
    int rc = encode_tensor_map(ptr, rows, cols, box_rows, &e.map);
    if (rc != LASER_OK) return rc;
    e.ptr = ptr;
    e.box_rows = box_rows;
    *out = &e.map;
    return LASER_OK;
}

int make_handle(const laser_probe_dims& dims, const laser_probe_options& opt, Handle** out) {
    DeviceInfo* di = nullptr;
    int rc = require_b200(&di);
    if (rc != LASER_OK) return rc;
    Handle* h = new (std::nothrow) Handle();
    if (!h) { g_last_error = "out of host memory"; return LASER_E_CUDA; }
    h->dims = dims;
    h->opt = opt;
    h->di = di;
    make_plan(dims, di->sms, opt.kernel_mode, &h->plan, &h->tail_plan);
    if (h->plan.mixed) fill_mixed_table(dims, h->plan, di->sms, h->mixed_tab);
    if (h->plan.flex) make_flex_plan(dims, di->sms, &h->plan, h->mixed_tab);
    const char* dbg = getenv("LASER_DEBUG");
    h->debug = dbg && dbg[0] && dbg[0] != '0';
    *out = h;
    return LASER_OK;
}

void free_handle(Handle* h) {
    if (!h) return;
    release_ctl(h->di, h->ctl);
    delete h;
}

// The decomposition of a call as the kernels see it (PlanDesc, probe_kernels.cuh).
PlanDesc plan_desc(const Handle* h, const int32_t* req_offsets) {
    const laser_probe_plan& pl = h->plan;
    PlanDesc d{};
    d.n_alloc = h->dims.N; d.R = h->dims.R; d.req_offsets = req_offsets;
    d.m_tiles = pl.m_tiles; d.rows_per_item = pl.tile_m; d.splits = pl.splits;
    d.total_tiles = ceil_div(h->dims.V, pl.tile_n);
    d.units = units_for(h->di, pl.cta_pair != 0);
    d.kind = pl.flex ? 3 : (pl.mixed ? 2 : (pl.m_tiles > 1 ? 1 : 0));
    if (pl.flex) memcpy(d.mixed_tab, h->mixed_tab, sizeof d.mixed_tab);
    if (pl.mixed) {
        d.tiles_pair = ceil_div(h->dims.V, pl.tile_n);
        d.sms = h->di->sms;
        memcpy(d.mixed_tab, h->mixed_tab, sizeof d.mixed_tab);
    }
    return d;
}

// Enqueue laser_probe_fused_kernel for the handle's dims (W has dims.V rows; v_offset localises
// token_ids); `tail` says what its last phase does.  role: 0 = the call's only fused kernel (plan
// h->plan); mixed schedule: 2 = the single-CTA tail-tile kernel (h->tail_plan), 1 = the pair kernel.
int launch_fused(Handle* h, int role, const void* hidden, const void* W, const int32_t* req_offsets,
                 const int32_t* token_ids, int v_offset, float4* ws, cudaStream_t stream, bool allow_pdl,
                 const TailParams& tail) {
    DeviceInfo* di = h->di;
    const laser_probe_plan& pl = role == 2 ? h->tail_plan : h->plan;
    const laser_probe_dims& dims = h->dims;
    const int N = dims.N;
    const bool pair = pl.cta_pair != 0;
    static const bool use_pdl = getenv("LASER_NO_PDL") == nullptr;
    if (!di->attr_set) {
        cudaError_t e = cudaFuncSetAttribute(laser_probe_fused_kernel<false>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(laser_probe_fused_kernel<true>,
                                     cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem);
        if (e != cudaSuccess) return set_cuda_error("cudaFuncSetAttribute", e);
        di->attr_set = true;
    }
    // Fewer than 128 rows in total: stage only the 8-row groups that hold rows.  TMA's zero fill of
    // out-of-range rows is slow (N = 8: 90 -> 75 us per step at the C2 shape without it).  The
    // other rows of the A tile keep whatever shared memory held; they feed TMEM lanes whose
    // statistics nobody reads (rows are independent).
    const int a_rows = N < kTileM ? round_up(N, 8) : kTileM;
    const int b_rows = pair ? pl.tile_n / 2 : pl.tile_n;   // W rows one CTA stages per tile
    const CUtensorMap *tm_h = nullptr, *tm_w = nullptr;
    int rc = handle_tensor_map(h->hid, 2, &h->hid_rr, hidden, N, dims.d, a_rows, &tm_h);
    if (rc != LASER_OK) return rc;
    // K-block-major W: k_blocks * V rows of 64 columns (one handle = one layout, so the cache key holds)
    const bool w_kblocked = h->opt.w_layout == LASER_W_KBLOCKED;
    if (w_kblocked) rc = handle_tensor_map(h->w, 4, &h->w_rr, W, dims.V * ceil_div(dims.d, kBlockK), kBlockK, b_rows, &tm_w);
    else rc = handle_tensor_map(h->w, 4, &h->w_rr, W, dims.V, dims.d, b_rows, &tm_w);
    if (rc != LASER_OK) return rc;

    FusedParams fp{};
    fp.w_kb_rows = w_kblocked ? dims.V : 0;
    fp.prefetch_slots = prefetch_slots_for(pl.stages);
    fp.n_alloc = N; fp.d = dims.d; fp.V = dims.V;
    fp.pd = plan_desc(h, req_offsets);
    fp.role = role;
    fp.grid_total = h->plan.grid;     // the fused tail exists only where one kernel makes the call
    fp.total_tiles = ceil_div(dims.V, pl.tile_n);
    fp.wait_first = (h->opt.overlap && !h->strict_inputs) ? 0 : 1;
    fp.early_w = (fp.wait_first && !h->opt.w_ordered) ? 1 : 0;   // W ahead of the wait unless it is produced on the stream
    fp.tile_n = pl.tile_n; fp.k_blocks = pl.k_blocks; fp.stages = pl.stages;
    fp.tail_cache = pl.tail_cache;
    fp.stage_bytes = static_cast<uint32_t>(kABytes + b_rows * 128);
    fp.tx_bytes = static_cast<uint32_t>((a_rows + b_rows) * 128);  // OOB rows are zero-filled and still counted
    // W is streamed once when a single token tile exists; with several token tiles the other
    // CTAs re-read the same rows from L2, so do not mark them evict-first.
    fp.w_policy = (h->plan.m_tiles == 1 && !h->plan.mixed) ? ptx::kEvictFirst : ptx::kEvictNormal;
    fp.ws = ws;
    fp.token_ids = token_ids;
    fp.v_offset = v_offset;

    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(pl.grid);
    cfg.blockDim = dim3(kFusedThreads);
    cfg.dynamicSmemBytes = static_cast<size_t>(pl.smem_bytes);
    cfg.stream = stream;
    // Programmatic dependent launch: the kernel may start while the previous kernel in the
    // stream is still running; it executes griddepcontrol.wait before it reads any per-call input
    // (strict) or before its first store (overlap), and always before it exits.
    cudaLaunchAttribute fattr[2];
    unsigned na = 0;
    if (use_pdl && allow_pdl) {
        fattr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        fattr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    // the two CTAs of a pair form a cluster (same TPC).  The single-CTA kernel of a mixed call is
    // launched as clusters of two as well - for placement only: its CTAs then fill whole TPCs and leave
    // whole TPCs to the pair kernel beside it (scattered over the TPCs they starve it of pairs).
    if (pair || (role == 2 && (pl.grid % 2) == 0)) {
        fattr[na].id = cudaLaunchAttributeClusterDimension;
        fattr[na].val.clusterDim.x = 2;
        fattr[na].val.clusterDim.y = 1;
        fattr[na].val.clusterDim.z = 1;
        ++na;
    }
    cfg.attrs = fattr;
    cfg.numAttrs = na;
#ifdef LASER_TIMELINE
    static int tl_launches = 0;      // debug build: one timeline slot per launch
    TailParams tail_tl = tail;
    tail_tl.tl_slot = tl_launches++;
    const TailParams& tail_arg = tail_tl;
#else
    const TailParams& tail_arg = tail;
#endif
    cudaError_t e = pair ? cudaLaunchKernelEx(&cfg, laser_probe_fused_kernel<true>, *tm_h, *tm_w, fp, tail_arg)
                         : cudaLaunchKernelEx(&cfg, laser_probe_fused_kernel<false>, *tm_h, *tm_w, fp, tail_arg);
    if (e != cudaSuccess) return set_cuda_error("launch laser_probe_fused_kernel", e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return LASER_OK;
}

// Enqueue laser_probe_flex_kernel (one launch: every decision about chunks and splits is the kernel's).
int launch_flex(Handle* h, const void* hidden, const void* W, const int32_t* req_offsets,
                const int32_t* token_ids, int v_offset, float4* ws, cudaStream_t stream, bool allow_pdl,
                const TailParams& tail) {
    DeviceInfo* di = h->di;
    const laser_probe_plan& pl = h->plan;
    const laser_probe_dims& dims = h->dims;
    static const bool use_pdl = getenv("LASER_NO_PDL") == nullptr;
    static bool attr_set[64] = {};
    int dev = static_cast<int>(di - g_dev);
    if (!attr_set[dev]) {
        cudaError_t e = cudaFuncSetAttribute(laser_probe_flex_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             kMaxDynSmem);
        if (e != cudaSuccess) return set_cuda_error("cudaFuncSetAttribute", e);
        attr_set[dev] = true;
    }
    const CUtensorMap* tm_w = nullptr;
    const bool w_kblocked = h->opt.w_layout == LASER_W_KBLOCKED;
    int rc = w_kblocked ? handle_tensor_map(h->w, 4, &h->w_rr, W, dims.V * ceil_div(dims.d, kBlockK), kBlockK, kTileM, &tm_w)
                        : handle_tensor_map(h->w, 4, &h->w_rr, W, dims.V, dims.d, kTileM, &tm_w);
    if (rc != LASER_OK) return rc;
    Handle::FlexEntry* fe = nullptr;
    for (auto& e : h->flex_hid)
        if (e.ptr == hidden) fe = &e;
    if (!fe) {
        fe = &h->flex_hid[h->flex_rr];
        h->flex_rr = (h->flex_rr + 1) % 2;
        fe->ptr = nullptr;
        for (int i = 0; i < kFlexMaps; ++i) {
            if (16 * (i + 1) > pl.flex_max_tok) { fe->maps.hid[i] = fe->maps.hid[0]; continue; }
            rc = encode_tensor_map(hidden, dims.N, dims.d, 8 * (i + 1), &fe->maps.hid[i]);
            if (rc != LASER_OK) return rc;
        }
        fe->ptr = hidden;
    }

    FusedParams fp{};
    fp.w_kb_rows = w_kblocked ? dims.V : 0;
    fp.prefetch_slots = prefetch_slots_for(pl.stages);
    fp.n_alloc = dims.N; fp.d = dims.d; fp.V = dims.V;
    fp.pd = plan_desc(h, req_offsets);
    fp.role = 0;
    fp.grid_total = pl.grid;
    fp.total_tiles = ceil_div(dims.V, kFlexVocabTile);
    fp.wait_first = (h->opt.overlap && !h->strict_inputs) ? 0 : 1;
    fp.tile_n = kFlexVocabTile; fp.k_blocks = pl.k_blocks; fp.stages = pl.stages;
    fp.tail_cache = pl.tail_cache;
    fp.stage_bytes = static_cast<uint32_t>(kABytes + (pl.flex_max_tok / 2) * 128);
    fp.tx_bytes = 0;       // depends on the chunk height: computed in the kernel
    fp.hint_C = pl.m_tiles; fp.hint_S = pl.splits;     // the dense decomposition (see the kernel)
    if (h->opt.w_ordered) fp.hint_C = 0;               // no guess, no W box ahead of the wait
    // several chunks re-read a W tile from L2 (side by side: chunk-fastest item order)
    fp.w_policy = pl.m_tiles == 1 && dims.N <= kFlexMaxTok ? ptx::kEvictFirst : ptx::kEvictNormal;
    fp.ws = ws;
    fp.token_ids = token_ids;
    fp.v_offset = v_offset;

    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(pl.grid);
    cfg.blockDim = dim3(kFusedThreads);
    cfg.dynamicSmemBytes = static_cast<size_t>(pl.smem_bytes);
    cfg.stream = stream;
    cudaLaunchAttribute fattr[2];
    unsigned na = 0;
    if (use_pdl && allow_pdl) {
        fattr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        fattr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    fattr[na].id = cudaLaunchAttributeClusterDimension;
    fattr[na].val.clusterDim.x = 2;
    fattr[na].val.clusterDim.y = 1;
    fattr[na].val.clusterDim.z = 1;
    ++na;
    cfg.attrs = fattr;
    cfg.numAttrs = na;
#ifdef LASER_TIMELINE
    static int tl_launches = 0;
    TailParams tail_tl = tail;
    tail_tl.tl_slot = tl_launches++;
    const TailParams& tail_arg = tail_tl;
#else
    const TailParams& tail_arg = tail;
#endif
    cudaError_t e = cudaLaunchKernelEx(&cfg, laser_probe_flex_kernel, fe->maps, *tm_w, fp, tail_arg);
    if (e != cudaSuccess) return set_cuda_error("launch laser_probe_flex_kernel", e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return LASER_OK;
}

// The fields of FinalizeParams that describe the fused kernels' workspace for the handle's dims.
FinalizeParams finalize_params(const Handle* h, bool run_fused, const int32_t* req_offsets) {
    FinalizeParams fz{};
    fz.n_alloc = h->dims.N; fz.R = h->dims.R;
    fz.pd = plan_desc(h, req_offsets);
    if (!run_fused) fz.pd.kind = 0;      // nothing was written: no request holds a row
    fz.req_offsets = req_offsets;
    fz.row_stride = 0; fz.split_stride = 1;    // packed records
    fz.wait_flags = nullptr; fz.epoch = 0; fz.a_offset = 0; fz.prob_mode = 0; fz.agg_mode = 0;
    return fz;
}

// One call's fused kernel(s): a single launch, or - mixed schedule - the single-CTA tail-tile kernel
// and, behind it under programmatic dependent launch, the pair kernel.  The two then run side by
// side (the CTAs either part does not need exit at once); nothing in one waits for the other, so a
// tool that serialises kernels only costs time.
int launch_call(Handle* h, const void* hidden, const void* W, const int32_t* req_offsets,
                const int32_t* token_ids, int v_offset, float4* ws, cudaStream_t stream, bool allow_pdl,
                const TailParams& tail) {
    if (h->plan.flex) return launch_flex(h, hidden, W, req_offsets, token_ids, v_offset, ws, stream, allow_pdl, tail);
    if (!h->plan.mixed) return launch_fused(h, 0, hidden, W, req_offsets, token_ids, v_offset, ws, stream, allow_pdl, tail);
    int rc = launch_fused(h, 2, hidden, W, req_offsets, token_ids, v_offset, ws, stream, allow_pdl, tail);
    if (rc != LASER_OK) return rc;
    return launch_fused(h, 1, hidden, W, req_offsets, token_ids, v_offset, ws, stream, true, tail);
}

// Enqueue laser_probe_finalize_kernel: blocks [0, R) aggregate, the rest mark padding rows.
int launch_finalize(const FinalizeParams& fz, cudaStream_t stream, bool pdl) {
    const int grid = fz.R + ceil_div(fz.n_alloc, kFinalizeThreads);
    if (grid <= 0) return LASER_OK;
    static const bool use_pdl = getenv("LASER_NO_PDL") == nullptr;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kFinalizeThreads);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    if (pdl && use_pdl) {
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
    }
    cudaError_t e = cudaLaunchKernelEx(&cfg, laser_probe_finalize_kernel, fz);
    if (e != cudaSuccess) return set_cuda_error("launch laser_probe_finalize_kernel", e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return LASER_OK;
}

// LASER_DEBUG=1: check the req_offsets precondition on the device ahead of the probe.
int launch_validate(const Handle* h, const int32_t* req_offsets, cudaStream_t stream) {
    if (!h->debug || h->dims.R <= 0) return LASER_OK;
    laser_probe_validate_kernel<<<1, 32, 0, stream>>>(req_offsets, h->dims.R, h->dims.N);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_cuda_error("launch laser_probe_validate_kernel", e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return LASER_OK;
}

// Does this call run its last phase inside the fused kernel?  Needs a control slot.
int want_fused_tail(Handle* h, cudaStream_t stream, bool* fused_tail) {
    *fused_tail = false;
    if (h->opt.tail == LASER_TAIL_SEPARATE) return LASER_OK;
    // AUTO with overlap: calls chained two deep gate each other's CTAs; the tail CTAs would hold SMs
    // the next call could be streaming on, so the second kernel (co-resident, tiny) is the faster form
    if (h->opt.tail == LASER_TAIL_AUTO && h->opt.overlap) return LASER_OK;
    // AUTO with many requests: the fused tail has at most kMaxFinalizers CTAs (see fused_tail), each of which
    // would take R / kMaxFinalizers requests one after the other; beyond two apiece the second kernel - a
    // block per request, a few microseconds behind kernels of hundreds - is the faster and the simpler form
    if (h->opt.tail == LASER_TAIL_AUTO && h->dims.R > 2 * kMaxFinalizers) return LASER_OK;
    if (!h->ctl) h->ctl = acquire_ctl(h->di, stream);
    if (h->ctl) { *fused_tail = true; return LASER_OK; }
    if (h->opt.tail == LASER_TAIL_FUSED) {
        g_last_error = "LASER_TAIL_FUSED: no control slot (first call under stream capture, or allocation failed)";
        return LASER_E_CUDA;
    }
    return LASER_OK;
}

int check_workspace(const Handle* h, const void* workspace, size_t workspace_bytes) {
    if (!workspace || workspace_bytes < workspace_bytes_for(h->plan) ||
        (reinterpret_cast<uintptr_t>(workspace) & 15))
        return LASER_E_WORKSPACE;
    return LASER_OK;
}

// ---- a1-a5 through a handle
int run_probe(Handle* h, const void* hidden, const void* W, const int32_t* req_offsets, const float* load,
              const laser_tau_params* tau_params, float* out_conf, int32_t* out_argmax, uint8_t* out_exit,
              void* workspace, size_t workspace_bytes, void* stream_v, float* out_tau_opt,
              float* out_pmax_opt, const int32_t* token_ids) {
    if (!tau_params) return LASER_E_NULL;
    if (!params_valid(tau_params)) return LASER_E_PARAMS;
    const int N = h->dims.N, R = h->dims.R;
    if (h->opt.prob_mode == LASER_PROB_TOKEN && N > 0 && !token_ids) return LASER_E_NULL;
    if (N == 0 && R == 0) return LASER_OK;
    if (N > 0 && (!hidden || !W || !out_argmax)) return LASER_E_NULL;
    if (R > 0 && (!req_offsets || !load || !out_conf || !out_exit)) return LASER_E_NULL;
    if ((reinterpret_cast<uintptr_t>(hidden) & 15) || (reinterpret_cast<uintptr_t>(W) & 15))
        return LASER_E_ALIGN;
    int rc = check_workspace(h, workspace, workspace_bytes);
    if (rc != LASER_OK) return rc;

    cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
    const bool run_fused = (N > 0 && R > 0);
    const bool prof = g_prof.on && g_prof.created && run_fused && g_prof.calls < kProfRing;
    const int prof_slot = g_prof.calls;

    FinalizeParams fz = finalize_params(h, run_fused, req_offsets);
    fz.agg_mode = h->opt.aggregate_mode;
    fz.prob_mode = h->opt.prob_mode;
    fz.ws = static_cast<const float4*>(workspace);
    fz.load = load;
    fz.out_conf = out_conf; fz.out_argmax = out_argmax; fz.out_exit = out_exit;
    fz.out_tau = out_tau_opt; fz.out_pmax = out_pmax_opt;
    fz.tau = to_dev(tau_params);

    bool fused_tail = false;
    if (run_fused) {
        rc = want_fused_tail(h, stream, &fused_tail);
        if (rc != LASER_OK) return rc;
        rc = launch_validate(h, req_offsets, stream);
        if (rc != LASER_OK) return rc;
        TailParams tail{};
        tail.kind = fused_tail ? 1 : 0;
        tail.ctl = h->ctl;
        tail.q.f = fz;
        if (prof) cudaEventRecord(g_prof.ev[prof_slot][0], stream);
        rc = launch_call(h, hidden, W, req_offsets,
                         h->opt.prob_mode == LASER_PROB_TOKEN ? token_ids : nullptr, 0,
                         static_cast<float4*>(workspace), stream, !prof && !h->debug, tail);
        if (rc != LASER_OK) return rc;
        if (prof) cudaEventRecord(g_prof.ev[prof_slot][1], stream);
    }
    if (!fused_tail) {
        // N == 0 with R > 0: every request is empty -> conf 0, exit 0, tau still defined.  Handled by
        // the same kernel (fz.R = R): req_offsets are all 0, no partials are read.
        rc = launch_finalize(fz, stream, run_fused && !prof);
        if (rc != LASER_OK) return rc;
    }
    if (prof) { cudaEventRecord(g_prof.ev[prof_slot][2], stream); g_prof.calls++; }
    return LASER_OK;
}

// ---- a1 + a2 over one vocabulary shard through a handle (dims.V = rows of the shard)
int run_partial(Handle* h, const void* hidden, const void* W_shard, const int32_t* req_offsets,
                const int32_t* token_ids_opt, int32_t v_offset, laser_row_stats* out_stats,
                const laser_probe_peers* peers_opt, void* workspace, size_t workspace_bytes, void* stream_v) {
    const int N = h->dims.N, R = h->dims.R;
    if (N > 0 && (!hidden || !W_shard)) return LASER_E_NULL;
    if (R > 0 && !req_offsets) return LASER_E_NULL;
    if ((reinterpret_cast<uintptr_t>(hidden) & 15) || (reinterpret_cast<uintptr_t>(W_shard) & 15) ||
        (reinterpret_cast<uintptr_t>(out_stats) & 15))
        return LASER_E_ALIGN;
    int rc = check_workspace(h, workspace, workspace_bytes);
    if (rc != LASER_OK) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
    const bool run_fused = (N > 0 && R > 0);

    ReduceParams rq{};
    rq.f = finalize_params(h, run_fused, req_offsets);
    rq.f.R = run_fused ? R : 0;            // R == 0: every row is padding -> neutral records
    rq.f.ws = static_cast<const float4*>(workspace);
    rq.f.a_offset = v_offset;
    rq.out_stats = reinterpret_cast<float4*>(out_stats);
    rq.rank = peers_opt ? peers_opt->rank : 0;
    rq.world = peers_opt ? peers_opt->world : 0;
    rq.epoch = peers_opt ? peers_opt->epoch : 0;
    for (int g = 0; g < rq.world; ++g) {
        rq.peer_stats[g] = reinterpret_cast<float4*>(peers_opt->peer_stats[g]);
        rq.peer_flags[g] = peers_opt->peer_flags[g];
    }
    bool fused_tail = false;
    if (run_fused) {
        rc = want_fused_tail(h, stream, &fused_tail);
        if (rc != LASER_OK) return rc;
        rc = launch_validate(h, req_offsets, stream);
        if (rc != LASER_OK) return rc;
        TailParams tail{};
        tail.kind = fused_tail ? 2 : 0;
        tail.ctl = h->ctl;
        tail.q = rq;
        rc = launch_call(h, hidden, W_shard, req_offsets, token_ids_opt, v_offset,
                         static_cast<float4*>(workspace), stream, !h->debug, tail);
        if (rc != LASER_OK) return rc;
        if (fused_tail) return LASER_OK;
    }
    if (N > 0) {
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(ceil_div(N, kFinalizeWarps));
        cfg.blockDim = dim3(kFinalizeThreads);
        cfg.stream = stream;
        cudaLaunchAttribute attr[1];
        static const bool use_pdl = getenv("LASER_NO_PDL") == nullptr;
        if (run_fused && use_pdl) {
            attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
            attr[0].val.programmaticStreamSerializationAllowed = 1;
            cfg.attrs = attr;
            cfg.numAttrs = 1;
        }
        cudaError_t e = cudaLaunchKernelEx(&cfg, laser_probe_reduce_kernel, rq);
        if (e != cudaSuccess) return set_cuda_error("launch laser_probe_reduce_kernel", e);
        g_launches.fetch_add(1, std::memory_order_relaxed);
    }
    if (peers_opt) {
        // Plain launch (full stream order): the reduce kernel's stores, remote ones included, have
        // been performed when this kernel starts; it publishes the epoch on every GPU.
        laser_probe_signal_kernel<<<1, 32, 0, stream>>>(rq);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return set_cuda_error("launch laser_probe_signal_kernel", e);
        g_launches.fetch_add(1, std::memory_order_relaxed);
    }
    return LASER_OK;
}

// Device-mapped address of a pinned host buffer (cached per handle), or nullptr if it is not mapped.
void* mapped_ptr(Handle* h, const void* host) {
    if (!host) return nullptr;
    for (auto& e : h->hm)
        if (e.h == host) return e.d;
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, host) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
    void* d = a.type == cudaMemoryTypeHost ? a.devicePointer : nullptr;
    if (d) {   // only successes are cached: a pageable buffer may be registered later
        Handle::HostMap& e = h->hm[h->hm_rr];
        h->hm_rr = (h->hm_rr + 1) % 8;
        e.h = host; e.d = d;
    }
    return d;
}

// ---- host buffers for the per-step tensors, through a handle
int run_host(Handle* h, const void* h_hidden, const void* W, const int32_t* h_req_offsets,
             const float* h_load, const laser_tau_params* tau_params, float* h_out_conf,
             int32_t* h_out_argmax, uint8_t* h_out_exit, void* workspace, size_t workspace_bytes,
             void* d_staging, size_t staging_bytes, void* stream_v, bool synchronize) {
    if (!tau_params) return LASER_E_NULL;
    const laser_probe_dims* dims = &h->dims;
    const int N = dims->N, R = dims->R;
    if (N == 0 && R == 0) return LASER_OK;
    if (!d_staging) return LASER_E_NULL;
    if (N > 0 && (!h_hidden || !h_out_argmax)) return LASER_E_NULL;
    if (R > 0 && (!h_req_offsets || !h_load || !h_out_conf || !h_out_exit)) return LASER_E_NULL;
    const Staging st = staging_layout(*dims);
    if (staging_bytes < st.total || (reinterpret_cast<uintptr_t>(d_staging) & 255)) return LASER_E_WORKSPACE;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
    uint8_t* base = static_cast<uint8_t*>(d_staging);
    cudaError_t e;
    // Rows >= req_offsets[R] are padding and never aggregated: copy the valid rows only (the offsets
    // are host memory here).  Out-of-range offsets fall back to all N rows.
    int n_copy = N;
    if (R > 0 && h_req_offsets[R] >= 0 && h_req_offsets[R] <= N) n_copy = h_req_offsets[R];
    else if (R == 0) n_copy = 0;
    if (n_copy > 0) {
        const size_t bytes = static_cast<size_t>(n_copy) * dims->d * 2;      // a multiple of 16 (d % 8 == 0)
        void* m_hidden = mapped_ptr(h, h_hidden);
        static const bool use_pdl = getenv("LASER_NO_PDL") == nullptr;
        if (m_hidden && (reinterpret_cast<uintptr_t>(m_hidden) & 15) == 0 && getenv("LASER_NO_STAGE_KERNEL") == nullptr) {
            // pinned + mapped: the staging kernel pulls the rows over PCIe as a link of the launch chain
            const int64_t n16 = static_cast<int64_t>(bytes / 16);
            int grid = static_cast<int>((n16 + kStageThreads * kStageInFlight - 1) / (kStageThreads * kStageInFlight));
            const int max_grid = 4 * h->di->sms;
            if (grid > max_grid) grid = max_grid;
            if (grid < 1) grid = 1;
            cudaLaunchConfig_t cfg{};
            cfg.gridDim = dim3(grid);
            cfg.blockDim = dim3(kStageThreads);
            cfg.stream = stream;
            cudaLaunchAttribute attr[1];
            if (use_pdl) {
                attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
                attr[0].val.programmaticStreamSerializationAllowed = 1;
                cfg.attrs = attr;
                cfg.numAttrs = 1;
            }
            e = cudaLaunchKernelEx(&cfg, laser_probe_stage_kernel, static_cast<const uint4*>(m_hidden),
                                   reinterpret_cast<uint4*>(base + st.hidden), n16);
            if (e != cudaSuccess) return set_cuda_error("launch laser_probe_stage_kernel", e);
            g_launches.fetch_add(1, std::memory_order_relaxed);
        } else {
            e = cudaMemcpyAsync(base + st.hidden, h_hidden, bytes, cudaMemcpyHostToDevice, stream);
            if (e != cudaSuccess) return set_cuda_error("H2D hidden", e);
        }
    }
    // Zero-copy for the small tensors: when req_offsets, load and the three outputs all live in
    // pinned, device-mapped host memory (cudaHostAlloc / cudaHostRegister / torch pin_memory), the
    // kernel's tail reads and writes them over PCIe directly and the call issues one copy (hidden)
    // instead of six.
    void* m_off = R > 0 ? mapped_ptr(h, h_req_offsets) : nullptr;
    void* m_load = R > 0 ? mapped_ptr(h, h_load) : nullptr;
    void* m_conf = R > 0 ? mapped_ptr(h, h_out_conf) : nullptr;
    void* m_exit = R > 0 ? mapped_ptr(h, h_out_exit) : nullptr;
    void* m_arg = N > 0 ? mapped_ptr(h, h_out_argmax) : nullptr;
    const bool zero_copy = (R == 0 || (m_off && m_load && m_conf && m_exit)) && (N == 0 || m_arg);
    int rc;
    // The staging buffer is written on this stream just ahead of the probe: an overlap = 1 handle must not let
    // the fused kernel read `hidden` (or the staged offsets / load) before that work has completed.
    h->strict_inputs = true;
    if (zero_copy) {
        rc = run_probe(h, base + st.hidden, W, static_cast<int32_t*>(m_off), static_cast<float*>(m_load),
                       tau_params, static_cast<float*>(m_conf), static_cast<int32_t*>(m_arg),
                       static_cast<uint8_t*>(m_exit), workspace, workspace_bytes, stream_v, nullptr, nullptr,
                       h->opt.token_ids);
        h->strict_inputs = false;
        if (rc != LASER_OK) return rc;
    } else {
        if (R > 0) {
            e = cudaMemcpyAsync(base + st.offsets, h_req_offsets, static_cast<size_t>(R + 1) * 4,
                                cudaMemcpyHostToDevice, stream);
            if (e != cudaSuccess) return set_cuda_error("H2D req_offsets", e);
            e = cudaMemcpyAsync(base + st.load, h_load, static_cast<size_t>(R) * 4, cudaMemcpyHostToDevice, stream);
            if (e != cudaSuccess) return set_cuda_error("H2D load", e);
        }
        rc = run_probe(h, base + st.hidden, W, reinterpret_cast<int32_t*>(base + st.offsets),
                       reinterpret_cast<float*>(base + st.load), tau_params,
                       reinterpret_cast<float*>(base + st.conf), reinterpret_cast<int32_t*>(base + st.argmax),
                       base + st.exit_, workspace, workspace_bytes, stream_v, nullptr, nullptr,
                       h->opt.token_ids);
        h->strict_inputs = false;
        if (rc != LASER_OK) return rc;
        if (R > 0) {
            e = cudaMemcpyAsync(h_out_conf, base + st.conf, static_cast<size_t>(R) * 4, cudaMemcpyDeviceToHost, stream);
            if (e != cudaSuccess) return set_cuda_error("D2H conf", e);
            e = cudaMemcpyAsync(h_out_exit, base + st.exit_, static_cast<size_t>(R), cudaMemcpyDeviceToHost, stream);
            if (e != cudaSuccess) return set_cuda_error("D2H exit", e);
        }
        if (N > 0) {
            e = cudaMemcpyAsync(h_out_argmax, base + st.argmax, static_cast<size_t>(N) * 4, cudaMemcpyDeviceToHost, stream);
            if (e != cudaSuccess) return set_cuda_error("D2H argmax", e);
        }
    }
    if (synchronize) {
        e = cudaStreamSynchronize(stream);
        if (e != cudaSuccess) return set_cuda_error("cudaStreamSynchronize", e);
    }
    return LASER_OK;
}

// ---------------------------------------------------------------------------------------- implicit handles
// The handle-less entry points (laser_probe_confidence and friends) keep a small per-thread cache of
// handles keyed by (device, dims, options, workspace): no lock, a linear scan of <= 16 entries.  The
// workspace is part of the key because calls that share a control slot must be stream-ordered, and
// the contract already forbids concurrent calls on one workspace.
struct ImplicitKey {
    int device;
    laser_probe_dims dims;
    int32_t agg, prob, mode, overlap, tail, w_layout, w_ordered;
    const void* workspace;
    bool operator==(const ImplicitKey& o) const {
        return device == o.device && dims.N == o.dims.N && dims.d == o.dims.d && dims.V == o.dims.V &&
               dims.R == o.dims.R && agg == o.agg && prob == o.prob && mode == o.mode &&
               overlap == o.overlap && tail == o.tail && w_layout == o.w_layout && w_ordered == o.w_ordered &&
               workspace == o.workspace;
    }
};
struct ImplicitCache {
    static constexpr int kCap = 16;
    struct Entry { ImplicitKey key; Handle* h; uint64_t stamp; };
    std::vector<Entry> entries;
    uint64_t clock = 0;
    ~ImplicitCache() { for (auto& e : entries) free_handle(e.h); }
};
thread_local ImplicitCache g_implicit;
std::atomic<uint64_t> g_cache_generation{0};      // bumped by laser_shutdown
thread_local uint64_t g_cache_seen = 0;

int implicit_handle(const laser_probe_dims& dims, const laser_probe_options& opt, const void* workspace,
                    Handle** out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); dev = -1; }
    ImplicitCache& c = g_implicit;
    const uint64_t gen = g_cache_generation.load(std::memory_order_relaxed);
    if (gen != g_cache_seen) {
        for (auto& e : c.entries) free_handle(e.h);
        c.entries.clear();
        g_cache_seen = gen;
    }
    const ImplicitKey key{dev, dims, opt.aggregate_mode, opt.prob_mode, opt.kernel_mode, opt.overlap, opt.tail,
                          opt.w_layout, opt.w_ordered, workspace};
    for (auto& e : c.entries)
        if (e.key == key) { e.stamp = ++c.clock; *out = e.h; return LASER_OK; }
    Handle* h = nullptr;
    int rc = make_handle(dims, opt, &h);
    if (rc != LASER_OK) return rc;
    h->opt.token_ids = nullptr;    // supplied per call
    if (static_cast<int>(c.entries.size()) >= ImplicitCache::kCap) {
        size_t lru = 0;
        for (size_t i = 1; i < c.entries.size(); ++i)
            if (c.entries[i].stamp < c.entries[lru].stamp) lru = i;
        free_handle(c.entries[lru].h);
        c.entries.erase(c.entries.begin() + static_cast<long>(lru));
    }
    c.entries.push_back({key, h, ++c.clock});
    *out = h;
    return LASER_OK;
}

}  // namespace

// ============================================================================================ static scratch
// Scratch of laser_probe_confidence_static (include/laser_probe.h): the per-row statistics records of
// the vocabulary splits, for callers that have no device workspace to give and cannot allocate one.
// Part of the device image: each GPU that loads this library's device code holds these bytes until the
// process exits.  In HOST code the name below is only a handle for the runtime's symbol table, not a
// device address - a kernel handed `laser_static_scratch` itself would fault (or, where the GPU can
// reach host memory, scribble over the wrong bytes).  static_scratch_ptr() asks the runtime for the
// array's address on the current device, once per device, and that address is what the kernels get.
static __device__ __align__(256) unsigned char laser_static_scratch[LASER_STATIC_SCRATCH_BYTES];

namespace {

std::mutex g_static_mu;
void* g_static_ptr[64] = {};       // device address of laser_static_scratch, per device ordinal

// Device address of the array on the CURRENT device (looked up on the first call per device, which
// should therefore be made outside any stream capture), or nullptr with g_last_error set.
void* static_scratch_ptr() {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) {
        (void)cudaGetLastError();
        g_last_error = "laser_probe_confidence_static: no current CUDA device";
        return nullptr;
    }
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, laser_static_scratch);
        if (e != cudaSuccess || !p) {
            (void)cudaGetLastError();
            g_last_error = std::string("cudaGetSymbolAddress(laser_static_scratch): ") + cudaGetErrorString(e);
            return nullptr;
        }
        g_static_ptr[dev] = p;
    }
    return g_static_ptr[dev];
}

}  // namespace

// ============================================================================================ ABI
extern "C" {

int laser_tau_params_default(laser_tau_params* out) {
    if (!out) return LASER_E_NULL;
    *out = laser_tau_params{0.95f, 0.04f, 1.0f, 10.0f, 0.88f, 0.97f};
    return LASER_OK;
}

size_t laser_probe_packed_w_bytes(int32_t V, int32_t d) {
    if (V <= 0 || d <= 0 || (d % 8) != 0) return 0;
    return static_cast<size_t>(ceil_div(d, kBlockK)) * static_cast<size_t>(V) * 128u;
}

int laser_probe_pack_w(const void* W, int32_t V, int32_t d, void* W_packed, void* stream_v) {
    if (!W || !W_packed) return LASER_E_NULL;
    if (V <= 0 || d <= 0 || (d % 8) != 0) return LASER_E_DIMS;
    if ((reinterpret_cast<uintptr_t>(W) & 15) || (reinterpret_cast<uintptr_t>(W_packed) & 15)) return LASER_E_ALIGN;
    DeviceInfo* di = nullptr;
    int rc = require_b200(&di);
    if (rc != LASER_OK) return rc;
    const int k_blocks = ceil_div(d, kBlockK);
    const int64_t total = static_cast<int64_t>(k_blocks) * V * 8;
    int64_t blocks = (total + 255) / 256;
    const int64_t cap = static_cast<int64_t>(di->sms) * 16;
    if (blocks > cap) blocks = cap;
    laser_probe_pack_w_kernel<<<static_cast<unsigned>(blocks), 256, 0, static_cast<cudaStream_t>(stream_v)>>>(
        static_cast<const uint4*>(W), static_cast<uint4*>(W_packed), V, d, k_blocks);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_cuda_error("launch laser_probe_pack_w_kernel", e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return LASER_OK;
}

int laser_probe_options_default(laser_probe_options* out) {
    if (!out) return LASER_E_NULL;
    *out = kDefaultOptions;
    return LASER_OK;
}

int laser_probe_plan_query_mode(const laser_probe_dims* dims, int kernel_mode, laser_probe_plan* plan) {
    if (!dims || !plan) return LASER_E_NULL;
    if (!dims_valid(dims)) return LASER_E_DIMS;
    if (kernel_mode < LASER_MODE_AUTO || kernel_mode > LASER_MODE_MIXED) return LASER_E_MODE;
    bool ok = false;
    DeviceInfo* di = current_device(&ok);
    make_plan(*dims, (ok && di) ? di->sms : kDefaultSMs, kernel_mode, plan, nullptr);
    return LASER_OK;
}

int laser_probe_mixed_query(const laser_probe_dims* dims, int32_t n_valid, laser_probe_mixed* out) {
    if (!dims || !out) return LASER_E_NULL;
    if (!dims_valid(dims) || n_valid < 0 || n_valid > dims->N) return LASER_E_DIMS;
    laser_probe_plan pl;
    int rc = laser_probe_plan_query_mode(dims, LASER_MODE_AUTO, &pl);
    if (rc != LASER_OK) return rc;
    memset(out, 0, sizeof *out);
    if (!pl.mixed) return LASER_OK;          // one single-CTA kernel: nothing is decided on the device
    const int m128 = ceil_div(n_valid, kTileM);
    if (m128 == 0) return LASER_OK;
    out->mixed = 1;
    if (m128 < kMixedTabMax) {
        const MixedChoice c = plan_mixed_host(m128, dims->V, dims->d, pl.tile_n, pl.tail_tile_n, pl.num_sms);
        const MixedPlan mp = mixed_unpack(mixed_pack(c.sched, c.u_tail, c.S_pair, c.S_tail), m128, pl.num_sms);
        out->schedule = c.sched; out->k_pair = mp.k_pair; out->j_single = mp.j_single;
        out->u_pair = mp.u_pair; out->u_single = mp.j_single > 0 ? mp.u_tail : 0;
        out->splits_pair = mp.S_pair; out->splits_single = mp.S_tail;
        out->model_us = static_cast<float>(c.time * 1e6);
    } else {
        const int k = (m128 + 1) / 2, up = pl.num_sms / 2 > 0 ? pl.num_sms / 2 : 1;
        out->schedule = 0; out->k_pair = k; out->u_pair = up;
        out->splits_pair = plan_splits(ceil_div(dims->V, pl.tile_n), k, up).splits;
    }
    return LASER_OK;
}

int laser_probe_flex_query(const laser_probe_dims* dims, int32_t n_valid, laser_probe_flex* out) {
    if (!dims || !out) return LASER_E_NULL;
    if (!dims_valid(dims) || n_valid < 0 || n_valid > kFlexMaxRows) return LASER_E_DIMS;
    bool ok = false;
    DeviceInfo* di = current_device(&ok);
    const FlexChoice c = plan_flex_host(n_valid, dims->V, (ok && di) ? di->sms : kDefaultSMs);
    out->chunks = c.C; out->n_tok = c.n_tok; out->splits = c.S; out->tiles_per_split = c.T;
    out->rounds = c.rounds; out->model_cost = static_cast<float>(c.cost);
    return LASER_OK;
}

int laser_probe_plan_query(const laser_probe_dims* dims, laser_probe_plan* plan) {
    return laser_probe_plan_query_mode(dims, LASER_MODE_AUTO, plan);
}

size_t laser_probe_workspace_bytes(const laser_probe_dims* dims) {
    // enough for every kernel_mode, so that one buffer serves every laser_probe_options setting
    size_t best = 0;
    for (int mode = LASER_MODE_AUTO; mode <= LASER_MODE_MIXED; ++mode) {
        laser_probe_plan pl;
        if (laser_probe_plan_query_mode(dims, mode, &pl) != LASER_OK) return 0;
        const size_t w = workspace_bytes_for(pl);
        if (w > best) best = w;
    }
    return best;
}

// ------------------------------------------------------------------------------ explicit handles
int laser_probe_handle_create(laser_probe_handle** out, const laser_probe_dims* dims,
                              const laser_probe_options* options) {
    if (!out || !dims) return LASER_E_NULL;
    *out = nullptr;
    if (!dims_valid(dims)) return LASER_E_DIMS;
    laser_probe_options opt = options ? *options : kDefaultOptions;
    int rc = options_valid(opt);
    if (rc != LASER_OK) return rc;
    Handle* h = nullptr;
    rc = make_handle(*dims, opt, &h);
    if (rc != LASER_OK) return rc;
    if (opt.tail != LASER_TAIL_SEPARATE)
        h->ctl = acquire_ctl(h->di, nullptr);   // may stay NULL: retried per call
    *out = h;
    return LASER_OK;
}

int laser_probe_handle_destroy(laser_probe_handle* h) {
    free_handle(h);
    return LASER_OK;
}

int laser_probe_handle_plan(const laser_probe_handle* h, laser_probe_plan* plan) {
    if (!h || !plan) return LASER_E_NULL;
    *plan = h->plan;
    const int fused = h->plan.mixed ? 2 : 1;    // fused kernels per call
    plan->kernel_launches = (h->opt.tail == LASER_TAIL_SEPARATE || !h->ctl ||
                             (h->opt.tail == LASER_TAIL_AUTO && (h->opt.overlap || h->dims.R > 2 * kMaxFinalizers)))
                                ? fused + 1 : fused;
    return LASER_OK;
}

size_t laser_probe_handle_workspace_bytes(const laser_probe_handle* h) {
    return h ? workspace_bytes_for(h->plan) : 0;
}

int laser_probe_handle_run(laser_probe_handle* h, const void* hidden, const void* W,
                           const int32_t* req_offsets, const float* load,
                           const laser_tau_params* tau_params, float* out_conf, int32_t* out_argmax,
                           uint8_t* out_exit, void* workspace, size_t workspace_bytes, void* stream,
                           float* out_tau_opt, float* out_pmax_opt) {
    if (!h) return LASER_E_NULL;
    return run_probe(h, hidden, W, req_offsets, load, tau_params, out_conf, out_argmax, out_exit, workspace,
                     workspace_bytes, stream, out_tau_opt, out_pmax_opt, h->opt.token_ids);
}

int laser_probe_handle_run_host(laser_probe_handle* h, const void* h_hidden, const void* W,
                                const int32_t* h_req_offsets, const float* h_load,
                                const laser_tau_params* tau_params, float* h_out_conf,
                                int32_t* h_out_argmax, uint8_t* h_out_exit, void* workspace,
                                size_t workspace_bytes, void* d_staging, size_t staging_bytes, void* stream,
                                int synchronize) {
    if (!h) return LASER_E_NULL;
    return run_host(h, h_hidden, W, h_req_offsets, h_load, tau_params, h_out_conf, h_out_argmax, h_out_exit,
                    workspace, workspace_bytes, d_staging, staging_bytes, stream, synchronize != 0);
}

// ------------------------------------------------------------------------------ handle-less forms
int laser_probe_confidence_opt(const void* hidden, const void* W, const int32_t* req_offsets,
                               const float* load, const laser_tau_params* tau_params,
                               float* out_conf, int32_t* out_argmax, uint8_t* out_exit,
                               const laser_probe_dims* dims, void* workspace,
                               size_t workspace_bytes, void* stream_v, float* out_tau_opt,
                               float* out_pmax_opt, const laser_probe_options* options) {
    if (!dims || !tau_params) return LASER_E_NULL;
    if (!dims_valid(dims)) return LASER_E_DIMS;
    if (!params_valid(tau_params)) return LASER_E_PARAMS;
    laser_probe_options opt = options ? *options : kDefaultOptions;
    int rc = options_valid(opt);
    if (rc != LASER_OK) return rc;
    const int N = dims->N, R = dims->R;
    if (opt.prob_mode == LASER_PROB_TOKEN && N > 0 && !opt.token_ids) return LASER_E_NULL;
    if (N == 0 && R == 0) return LASER_OK;
    if (N > 0 && (!hidden || !W || !out_argmax)) return LASER_E_NULL;
    if (R > 0 && (!req_offsets || !load || !out_conf || !out_exit)) return LASER_E_NULL;
    if ((reinterpret_cast<uintptr_t>(hidden) & 15) || (reinterpret_cast<uintptr_t>(W) & 15))
        return LASER_E_ALIGN;
    Handle* h = nullptr;
    rc = implicit_handle(*dims, opt, workspace, &h);
    if (rc != LASER_OK) return rc;
    return run_probe(h, hidden, W, req_offsets, load, tau_params, out_conf, out_argmax, out_exit, workspace,
                     workspace_bytes, stream_v, out_tau_opt, out_pmax_opt, opt.token_ids);
}

int laser_probe_confidence_agg(const void* hidden, const void* W, const int32_t* req_offsets,
                               const float* load, const laser_tau_params* tau_params,
                               float* out_conf, int32_t* out_argmax, uint8_t* out_exit,
                               const laser_probe_dims* dims, void* workspace,
                               size_t workspace_bytes, void* stream, float* out_tau_opt,
                               float* out_pmax_opt, int aggregate_mode) {
    laser_probe_options opt = kDefaultOptions;
    opt.aggregate_mode = aggregate_mode;
    return laser_probe_confidence_opt(hidden, W, req_offsets, load, tau_params, out_conf, out_argmax,
                                      out_exit, dims, workspace, workspace_bytes, stream, out_tau_opt,
                                      out_pmax_opt, &opt);
}

int laser_probe_confidence(const void* hidden, const void* W, const int32_t* req_offsets,
                           const float* load, const laser_tau_params* tau_params, float* out_conf,
                           int32_t* out_argmax, uint8_t* out_exit, const laser_probe_dims* dims,
                           void* workspace, size_t workspace_bytes, void* stream,
                           float* out_tau_opt, float* out_pmax_opt) {
    return laser_probe_confidence_opt(hidden, W, req_offsets, load, tau_params, out_conf, out_argmax,
                                      out_exit, dims, workspace, workspace_bytes, stream, out_tau_opt,
                                      out_pmax_opt, nullptr);
}

// ------------------------------------------------------------------------------ no device allocation
// laser_probe_confidence_opt with the library's static array as the workspace and the separate tail (no
// control block).  Between entry and return: no cudaMalloc / cudaFree / memset / memcpy; host-side `new`
// of the implicit handle on the first call per (dims, options) only.
int laser_probe_confidence_static(const void* hidden, const void* W, const int32_t* req_offsets,
                                  const float* load, const laser_tau_params* tau_params,
                                  float* out_conf, int32_t* out_argmax, uint8_t* out_exit,
                                  const laser_probe_dims* dims, void* stream_v, float* out_tau_opt,
                                  float* out_pmax_opt, const laser_probe_options* options) {
    if (!dims || !tau_params) return LASER_E_NULL;
    if (!dims_valid(dims)) return LASER_E_DIMS;
    if (!params_valid(tau_params)) return LASER_E_PARAMS;
    laser_probe_options opt = options ? *options : kDefaultOptions;
    int rc = options_valid(opt);
    if (rc != LASER_OK) return rc;
    opt.tail = LASER_TAIL_SEPARATE;        // the fused tail needs the cudaMalloc'ed control block
    const int N = dims->N, R = dims->R;
    if (opt.prob_mode == LASER_PROB_TOKEN && N > 0 && !opt.token_ids) return LASER_E_NULL;
    if (N == 0 && R == 0) return LASER_OK;
    if (N > 0 && (!hidden || !W || !out_argmax)) return LASER_E_NULL;
    if (R > 0 && (!req_offsets || !load || !out_conf || !out_exit)) return LASER_E_NULL;
    if ((reinterpret_cast<uintptr_t>(hidden) & 15) || (reinterpret_cast<uintptr_t>(W) & 15))
        return LASER_E_ALIGN;
    // the documented rule: what laser_probe_workspace_bytes says (any kernel_mode) must fit the array
    const size_t need = laser_probe_workspace_bytes(dims);
    if (need == 0) return LASER_E_DIMS;
    if (need > static_cast<size_t>(LASER_STATIC_SCRATCH_BYTES)) {
        char buf[256];
        snprintf(buf, sizeof buf,
                 "laser_probe_confidence_static: N=%d d=%d V=%d R=%d needs %zu bytes of scratch, the built-in "
                 "array holds %u (LASER_STATIC_SCRATCH_BYTES); use laser_probe_confidence with a workspace",
                 dims->N, dims->d, dims->V, dims->R, need, static_cast<unsigned>(LASER_STATIC_SCRATCH_BYTES));
        g_last_error = buf;
        return LASER_E_STATIC_LIMIT;
    }
    DeviceInfo* di = nullptr;
    rc = require_b200(&di);
    if (rc != LASER_OK) return rc;
    void* scratch = static_scratch_ptr();
    if (!scratch) return LASER_E_CUDA;
    Handle* h = nullptr;
    rc = implicit_handle(*dims, opt, scratch, &h);
    if (rc != LASER_OK) return rc;
    return run_probe(h, hidden, W, req_offsets, load, tau_params, out_conf, out_argmax, out_exit, scratch,
                     static_cast<size_t>(LASER_STATIC_SCRATCH_BYTES), stream_v, out_tau_opt, out_pmax_opt,
                     opt.token_ids);
}

// ------------------------------------------------------------------------------ vocabulary-parallel
int laser_probe_partial(const void* hidden, const void* W_shard, const int32_t* req_offsets,
                        const int32_t* token_ids_opt, const laser_probe_dims* dims, int32_t v_offset,
                        laser_row_stats* out_stats, const laser_probe_peers* peers_opt,
                        void* workspace, size_t workspace_bytes, void* stream_v,
                        const laser_probe_options* options) {
    if (!dims) return LASER_E_NULL;
    if (!dims_valid(dims) || v_offset < 0) return LASER_E_DIMS;
    if (!out_stats && !peers_opt) return LASER_E_NULL;
    if (peers_opt) {
        const laser_probe_peers& pe = *peers_opt;
        if (pe.world < 1 || pe.world > LASER_MAX_PEERS || pe.rank < 0 || pe.rank >= pe.world || pe.epoch == 0)
            return LASER_E_PARAMS;
        for (int g = 0; g < pe.world; ++g)
            if (!pe.peer_stats[g] || !pe.peer_flags[g]) return LASER_E_NULL;
    }
    laser_probe_options opt = options ? *options : kDefaultOptions;
    int rc = options_valid(opt);
    if (rc != LASER_OK) return rc;
    const int N = dims->N, R = dims->R;
    if (N > 0 && (!hidden || !W_shard)) return LASER_E_NULL;
    if (R > 0 && !req_offsets) return LASER_E_NULL;
    if ((reinterpret_cast<uintptr_t>(hidden) & 15) || (reinterpret_cast<uintptr_t>(W_shard) & 15) ||
        (reinterpret_cast<uintptr_t>(out_stats) & 15))
        return LASER_E_ALIGN;
    opt.aggregate_mode = LASER_AGG_MEAN; opt.prob_mode = LASER_PROB_MAX;   // not part of the partial
    Handle* h = nullptr;
    rc = implicit_handle(*dims, opt, workspace, &h);
    if (rc != LASER_OK) return rc;
    return run_partial(h, hidden, W_shard, req_offsets, token_ids_opt, v_offset, out_stats, peers_opt,
                       workspace, workspace_bytes, stream_v);
}

int laser_probe_combine(const laser_row_stats* stats, int32_t G, const int32_t* req_offsets,
                        const float* load, const laser_tau_params* tau_params, float* out_conf,
                        int32_t* out_argmax, uint8_t* out_exit, const laser_probe_dims* dims,
                        void* stream_v, float* out_tau_opt, float* out_pmax_opt,
                        const laser_probe_options* options, const uint32_t* wait_flags_opt,
                        uint32_t epoch) {
    if (!dims || !tau_params) return LASER_E_NULL;
    if (!dims_valid(dims)) return LASER_E_DIMS;
    if (G < 1 || G > LASER_MAX_PEERS) return LASER_E_DIMS;
    if (!params_valid(tau_params)) return LASER_E_PARAMS;
    laser_probe_options opt = options ? *options : kDefaultOptions;
    int rc = options_valid(opt);
    if (rc != LASER_OK) return rc;
    const int N = dims->N, R = dims->R;
    if (N == 0 && R == 0) return LASER_OK;
    if (N > 0 && (!stats || !out_argmax)) return LASER_E_NULL;
    if (R > 0 && (!req_offsets || !load || !out_conf || !out_exit)) return LASER_E_NULL;
    if (reinterpret_cast<uintptr_t>(stats) & 15) return LASER_E_ALIGN;
    DeviceInfo* di = nullptr;
    rc = require_b200(&di);
    if (rc != LASER_OK) return rc;
    FinalizeParams fz{};
    fz.n_alloc = N; fz.R = R;
    fz.pd.kind = 0; fz.pd.n_alloc = N; fz.pd.R = R; fz.pd.req_offsets = req_offsets;
    fz.pd.m_tiles = 1; fz.pd.rows_per_item = kTileM; fz.pd.splits = G;
    fz.agg_mode = opt.aggregate_mode;
    fz.prob_mode = opt.prob_mode;
    fz.a_offset = 0;
    fz.ws = reinterpret_cast<const float4*>(stats);
    fz.row_stride = 1; fz.split_stride = N;
    fz.wait_flags = wait_flags_opt; fz.epoch = epoch;
    fz.req_offsets = req_offsets; fz.load = load;
    fz.out_conf = out_conf; fz.out_argmax = out_argmax; fz.out_exit = out_exit;
    fz.out_tau = out_tau_opt; fz.out_pmax = out_pmax_opt;
    fz.tau = to_dev(tau_params);
    // Programmatic dependent launch: the blocks become resident while the kernel ahead (the partial, or a
    // collective that never triggers early - then this is an ordinary launch) still runs; they read
    // offsets / load, wait for its completion (griddepcontrol.wait), then for the peers' flags.
    return launch_finalize(fz, static_cast<cudaStream_t>(stream_v), true);
}

size_t laser_probe_staging_bytes(const laser_probe_dims* dims) {
    if (!dims_valid(dims)) return 0;
    return staging_layout(*dims).total;
}

int laser_probe_confidence_host_async(const void* h_hidden, const void* W, const int32_t* h_req_offsets,
                                      const float* h_load, const laser_tau_params* tau_params,
                                      float* h_out_conf, int32_t* h_out_argmax, uint8_t* h_out_exit,
                                      const laser_probe_dims* dims, void* workspace,
                                      size_t workspace_bytes, void* d_staging, size_t staging_bytes,
                                      void* stream_v) {
    if (!dims || !tau_params) return LASER_E_NULL;
    if (!dims_valid(dims)) return LASER_E_DIMS;
    if (dims->N == 0 && dims->R == 0) return LASER_OK;
    Handle* h = nullptr;
    int rc = implicit_handle(*dims, kDefaultOptions, workspace, &h);
    if (rc != LASER_OK) return rc;
    return run_host(h, h_hidden, W, h_req_offsets, h_load, tau_params, h_out_conf, h_out_argmax, h_out_exit,
                    workspace, workspace_bytes, d_staging, staging_bytes, stream_v, false);
}

int laser_probe_confidence_host(const void* h_hidden, const void* W, const int32_t* h_req_offsets,
                                const float* h_load, const laser_tau_params* tau_params,
                                float* h_out_conf, int32_t* h_out_argmax, uint8_t* h_out_exit,
                                const laser_probe_dims* dims, void* workspace,
                                size_t workspace_bytes, void* d_staging, size_t staging_bytes,
                                void* stream_v) {
    if (!dims || !tau_params) return LASER_E_NULL;
    if (!dims_valid(dims)) return LASER_E_DIMS;
    if (dims->N == 0 && dims->R == 0) return LASER_OK;
    Handle* h = nullptr;
    int rc = implicit_handle(*dims, kDefaultOptions, workspace, &h);
    if (rc != LASER_OK) return rc;
    return run_host(h, h_hidden, W, h_req_offsets, h_load, tau_params, h_out_conf, h_out_argmax, h_out_exit,
                    workspace, workspace_bytes, d_staging, staging_bytes, stream_v, true);
}

int laser_tau_from_load(const float* load, int32_t R, const laser_tau_params* tau_params, float* out_tau) {
    if (!tau_params || (R > 0 && (!load || !out_tau))) return LASER_E_NULL;
    if (R < 0) return LASER_E_DIMS;
    if (!params_valid(tau_params)) return LASER_E_PARAMS;
    const TauParamsDev t = to_dev(tau_params);
    for (int32_t r = 0; r < R; ++r) out_tau[r] = tau_eval(load[r], t);
    return LASER_OK;
}

int laser_ema_update(float* lbar, const float* L, int32_t R, float alpha) {
    if (R > 0 && (!lbar || !L)) return LASER_E_NULL;
    if (R < 0) return LASER_E_DIMS;
    if (!(alpha >= 0.f && alpha <= 1.f)) return LASER_E_PARAMS;
    for (int32_t r = 0; r < R; ++r) lbar[r] = alpha * L[r] + (1.f - alpha) * lbar[r];
    return LASER_OK;
}

int laser_budget_params_default(laser_budget_params* out) {
    if (!out) return LASER_E_NULL;
    *out = laser_budget_params{10.0, 2.0, 0.6, 1.5, 50.0, 275.0, 10.0};
    return LASER_OK;
}

int laser_allocate_budget(const int32_t* prompt_tokens, const float* L, int32_t R,
                          const laser_budget_params* q, int32_t* out_budget) {
    if (!q || (R > 0 && (!prompt_tokens || !L || !out_budget))) return LASER_E_NULL;
    if (R < 0) return LASER_E_DIMS;
    if (!(q->p_max > q->p_min) || !(q->f_max >= q->f_min) || !(q->l_target > 0.0)) return LASER_E_PARAMS;
    for (int32_t r = 0; r < R; ++r) {
        // Eq. 7: difficulty factor from the prompt length, clipped to [f_min, f_max]
        double f_diff = q->f_min + (static_cast<double>(prompt_tokens[r]) - q->p_min) / (q->p_max - q->p_min) *
                                       (q->f_max - q->f_min);
        f_diff = f_diff < q->f_min ? q->f_min : (f_diff > q->f_max ? q->f_max : f_diff);
        // Eq. 8: load factor min(1, L_target / max(1, L(t)))
        const double den = L[r] > 1.f ? static_cast<double>(L[r]) : 1.0;
        double f_load = q->l_target / den;
        f_load = f_load < 1.0 ? f_load : 1.0;
        // Eq. 6; the floor is that of the real-number product: a binary product that lands within
        // LASER_BUDGET_FLOOR_EPS below an integer (|p| = 100: 10 * 0.8 = 7.999...) is that integer
        double b = std::floor(q->b_base * f_diff * f_load + LASER_BUDGET_FLOOR_EPS);
        if (b < q->b_min) b = q->b_min;
        out_budget[r] = static_cast<int32_t>(b);
    }
    return LASER_OK;
}

const char* laser_status_string(int status) {
    switch (status) {
        case LASER_OK: return "ok";
        case LASER_E_NULL: return "required pointer is NULL";
        case LASER_E_DIMS: return "invalid dimensions (need d > 0, d % 8 == 0, V > 0, N >= 0, R >= 0)";
        case LASER_E_ALIGN: return "hidden / W must be 16-byte aligned";
        case LASER_E_PARAMS: return "invalid parameters";
        case LASER_E_WORKSPACE: return "workspace / staging buffer missing, misaligned or too small";
        case LASER_E_ARCH: return "device is not sm_100 (B200); this library has no fallback path";
        case LASER_E_CUDA: return "CUDA call failed (see laser_last_error)";
        case LASER_E_MODE: return "unknown aggregate / probability / kernel / tail mode or option";
        case LASER_E_STATIC_LIMIT:
            return "batch needs more scratch than the library's built-in array holds (see laser_last_error)";
        default: return "unknown status";
    }
}

int laser_profile_enable(int on) {
    if (on && !g_prof.created) {
        for (int i = 0; i < kProfRing; ++i)
            for (int j = 0; j < 3; ++j) {
                cudaError_t e = cudaEventCreate(&g_prof.ev[i][j]);
                if (e != cudaSuccess) return set_cuda_error("cudaEventCreate", e);
            }
        g_prof.created = true;
    }
    g_prof.on = on != 0;
    g_prof.calls = 0;
    return LASER_OK;
}

int laser_profile_read(float* ms_fused_sum, float* ms_finalize_sum, int32_t* calls) {
    if (!ms_fused_sum || !ms_finalize_sum || !calls) return LASER_E_NULL;
    *ms_fused_sum = 0.f; *ms_finalize_sum = 0.f; *calls = g_prof.calls;
    if (!g_prof.created || g_prof.calls == 0) return LASER_OK;
    cudaError_t e = cudaEventSynchronize(g_prof.ev[g_prof.calls - 1][2]);
    if (e != cudaSuccess) return set_cuda_error("cudaEventSynchronize", e);
    for (int i = 0; i < g_prof.calls; ++i) {
        float a = 0.f, b = 0.f;
        cudaEventElapsedTime(&a, g_prof.ev[i][0], g_prof.ev[i][1]);
        cudaEventElapsedTime(&b, g_prof.ev[i][1], g_prof.ev[i][2]);
        *ms_fused_sum += a; *ms_finalize_sum += b;
    }
    g_prof.calls = 0;
    return LASER_OK;
}

#ifdef LASER_TIMELINE
int laser_debug_timeline_read(unsigned long long* out) {   // [8][160][8]
    return cudaMemcpyFromSymbol(out, laser::g_timeline, sizeof(unsigned long long) * 8 * 160 * 8) == cudaSuccess ? 0 : -7;
}
#endif

const char* laser_last_error(void) { return g_last_error.c_str(); }

uint64_t laser_kernel_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

int laser_shutdown(void) {
    // implicit handles are per thread: this thread's go now, every other thread drops its own at its next call
    const uint64_t gen = g_cache_generation.fetch_add(1, std::memory_order_relaxed) + 1;
    for (auto& e : g_implicit.entries) free_handle(e.h);
    g_implicit.entries.clear();
    g_cache_seen = gen;
    // a device's control block is freed once no handle - explicit, or another thread's implicit one - holds a
    // slot of it (the caller has made sure that the work enqueued through the handles has completed); the next
    // fused-tail call allocates a new one
    std::lock_guard<std::mutex> lk(g_mu);
    for (DeviceInfo& d : g_dev) {
        if (d.ctl_base && static_cast<int>(d.ctl_free.size()) == kCtlSlots) {
            if (cudaFree(d.ctl_base) != cudaSuccess) (void)cudaGetLastError();
            d.ctl_base = nullptr;
            d.ctl_free.clear();
        }
    }
    return LASER_OK;
}

}  // extern "C"
