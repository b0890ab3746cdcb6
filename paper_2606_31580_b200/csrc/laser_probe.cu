// laser_probe.cu — host side of the C ABI declared in include/laser_probe.h: argument validation,
// launch planning, TMA descriptor encoding (driver entry point fetched through the runtime, no
// -lcuda), and the two kernel launches.  No device allocation, no host<->device synchronisation
// (except in the explicit *_host entry point), no fallback path.
#include "../../include/laser_probe.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <unordered_map>

#include "probe_kernels.cuh"

namespace {

using namespace laser;

thread_local std::string g_last_error;
std::atomic<uint64_t> g_launches{0};

// Optional per-kernel timing (bench / profiling only): when enabled on this thread, every call
// records events before the fused kernel, between the kernels and after the finalize kernel.
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

int set_cuda_error(const char* what, cudaError_t e) {
    g_last_error = std::string(what) + ": " + cudaGetErrorString(e);
    return LASER_E_CUDA;
}

// ---------------------------------------------------------------------------------------- device
struct DeviceInfo {
    bool queried = false, ok = false;
    int sms = kDefaultSMs, cc_major = 0, cc_minor = 0;
    bool attr_set = false;
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
    std::lock_guard<std::mutex> lk(g_mu);
    DeviceInfo& d = g_dev[dev];
    if (!d.queried) {
        d.queried = true;
        d.ok = cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess &&
               cudaDeviceGetAttribute(&d.cc_major, cudaDevAttrComputeCapabilityMajor, dev) == cudaSuccess &&
               cudaDeviceGetAttribute(&d.cc_minor, cudaDevAttrComputeCapabilityMinor, dev) == cudaSuccess;
        if (!d.ok) (void)cudaGetLastError();
    }
    *cuda_ok = d.ok;
    return &d;
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

std::atomic<int> g_force_mode{LASER_MODE_AUTO};
std::atomic<int> g_overlap{0};   // strict stream order unless the caller opts in

void make_plan(const laser_probe_dims& dm, int num_sms, laser_probe_plan* pl) {
    // CTA pairs (tcgen05 cta_group::2, M = 256) when there is more than one 128-row token tile: each
    // W tile then enters a pair's shared memory once instead of once per token tile and one issuing
    // thread feeds two SMs' tensor cores (measured +10..17 % for N >= 256).  An odd count of 128-row
    // tiles makes the pair kernel compute one padding tile; that costs more than the pair gains
    // until there are about ten tiles (measured: N = 384 and 640 are faster on single CTAs).
    const int mode = g_force_mode.load(std::memory_order_relaxed);
    const int t128 = ceil_div(dm.N, kTileM);
    const bool auto_pair = t128 >= 2 && ((t128 % 2) == 0 || t128 >= 10);
    const bool pair = mode == LASER_MODE_PAIR || (mode == LASER_MODE_AUTO && auto_pair);
    const int tile_m = pair ? 2 * kTileM : kTileM;
    const int units = pair ? (num_sms / 2 > 0 ? num_sms / 2 : 1) : num_sms;
    int S, T, BN;
    plan_variant(dm, units, tile_m, pair ? 32 : 16, &S, &T, &BN);   // fixes the tile height BN
    pl->num_sms = num_sms;
    pl->m_tiles = dm.N > 0 ? ceil_div(dm.N, tile_m) : 1;
    // The deal of tiles to units comes from the function the kernels also use: with padding rows in
    // the batch they re-plan on the device for the token items that hold rows (same BN).
    const int total_tiles = ceil_div(dm.V, BN);
    const SplitPlan sp = plan_splits(total_tiles, pl->m_tiles, units);
    S = sp.splits; T = sp.T;
    int ws_splits = S;
    for (int m = 1; m < pl->m_tiles; ++m) {
        const int sm = plan_splits(total_tiles, m, units).splits;
        if (sm > ws_splits) ws_splits = sm;
    }
    pl->ws_splits = ws_splits;
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
    pl->smem_bytes = stages * stage_bytes + kSmemSlack;
    pl->kernel_launches = 2;
    pl->tile_m = tile_m;
    pl->cta_pair = pair ? 1 : 0;
}

size_t workspace_bytes_for(const laser_probe_plan& pl) {
    size_t b = static_cast<size_t>(16) * pl.ws_splits * pl.m_tiles * pl.tile_m;
    return b < 16 ? 16 : b;
}

// ---------------------------------------------------------------------------------------- TMA maps
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;

struct MapKey {
    const void* ptr;
    int rows, cols, box_rows;
    bool operator==(const MapKey& o) const {
        return ptr == o.ptr && rows == o.rows && cols == o.cols && box_rows == o.box_rows;
    }
};
struct MapKeyHash {
    size_t operator()(const MapKey& k) const {
        size_t h = reinterpret_cast<size_t>(k.ptr);
        h ^= (static_cast<size_t>(k.rows) * 0x9E3779B97F4A7C15ull) ^ (static_cast<size_t>(k.cols) << 20) ^
             (static_cast<size_t>(k.box_rows) << 44);
        return h;
    }
};
std::unordered_map<MapKey, CUtensorMap, MapKeyHash> g_maps;

// bf16 [rows, cols] row-major; box = 64 columns (128 B, the swizzle span) x box_rows rows.
int get_tensor_map(const void* ptr, int rows, int cols, int box_rows, CUtensorMap* out) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) {
            (void)cudaGetLastError();
            g_last_error = "cudaGetDriverEntryPoint(cuTensorMapEncodeTiled) failed";
            return LASER_E_CUDA;
        }
        g_encode = reinterpret_cast<EncodeTiledFn>(fn);
    }
    const MapKey key{ptr, rows, cols, box_rows};
    auto it = g_maps.find(key);
    if (it != g_maps.end()) { *out = it->second; return LASER_OK; }
    const cuuint64_t gdim[2] = {static_cast<cuuint64_t>(cols), static_cast<cuuint64_t>(rows)};
    const cuuint64_t gstride[1] = {static_cast<cuuint64_t>(cols) * 2};
    const cuuint32_t box[2] = {static_cast<cuuint32_t>(kBlockK), static_cast<cuuint32_t>(box_rows)};
    const cuuint32_t estr[2] = {1, 1};
    CUtensorMap m;
    CUresult r = g_encode(&m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), gdim,
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
    if (g_maps.size() > 256) g_maps.clear();
    g_maps.emplace(key, m);
    *out = m;
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

int options_valid(const laser_probe_options& o, int N) {
    if (o.aggregate_mode < LASER_AGG_MEAN || o.aggregate_mode > LASER_AGG_MIN) return LASER_E_MODE;
    if (o.prob_mode < LASER_PROB_MAX || o.prob_mode > LASER_PROB_TOKEN) return LASER_E_MODE;
    if (o.prob_mode == LASER_PROB_TOKEN && N > 0 && !o.token_ids) return LASER_E_NULL;
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

int units_for(const DeviceInfo* di, bool pair) { return pair ? (di->sms / 2 > 0 ? di->sms / 2 : 1) : di->sms; }

// Enqueue laser_probe_fused_kernel for `dims` (W has dims.V rows; v_offset localises token_ids).
int launch_fused(DeviceInfo* di, const laser_probe_plan& pl, const void* hidden, const void* W,
                 const int32_t* req_offsets, const laser_probe_dims& dims, const int32_t* token_ids,
                 int v_offset, float4* ws, cudaStream_t stream, bool allow_pdl) {
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
    CUtensorMap tm_h, tm_w;
    // Fewer than 128 rows in total: stage only the 8-row groups that hold rows.  TMA's zero fill of
    // out-of-range rows is slow (N = 8: 90 -> 75 us per step at the C2 shape without it).  The
    // other rows of the A tile keep whatever shared memory held; they feed TMEM lanes whose
    // statistics nobody reads (rows are independent).
    const int a_rows = N < kTileM ? round_up(N, 8) : kTileM;
    int rc = get_tensor_map(hidden, N, dims.d, a_rows, &tm_h);
    if (rc != LASER_OK) return rc;
    const int b_rows = pair ? pl.tile_n / 2 : pl.tile_n;   // W rows one CTA stages per tile
    rc = get_tensor_map(W, dims.V, dims.d, b_rows, &tm_w);
    if (rc != LASER_OK) return rc;

    FusedParams fp;
    fp.n_alloc = N; fp.d = dims.d; fp.V = dims.V;
    fp.m_tiles = pl.m_tiles; fp.splits = pl.ws_splits; fp.tiles_per_split = pl.tiles_per_split;
    fp.req_offsets = req_offsets; fp.R = dims.R;
    fp.total_tiles = ceil_div(dims.V, pl.tile_n);
    fp.units = units_for(di, pair);
    fp.replan = pl.m_tiles > 1 ? 1 : 0;
    fp.wait_first = g_overlap.load(std::memory_order_relaxed) ? 0 : 1;
    fp.tile_n = pl.tile_n; fp.k_blocks = pl.k_blocks; fp.stages = pl.stages;
    fp.work_items = pl.work_items; fp.n_pad = pl.m_tiles * pl.tile_m;
    fp.stage_bytes = static_cast<uint32_t>(kABytes + b_rows * 128);
    fp.tx_bytes = static_cast<uint32_t>((a_rows + b_rows) * 128);  // OOB rows are zero-filled and still counted
    // W is streamed once when a single token tile exists; with several token tiles the other
    // CTAs re-read the same rows from L2, so do not mark them evict-first.
    fp.w_policy = (pl.m_tiles == 1) ? ptx::kEvictFirst : ptx::kEvictNormal;
    fp.ws = ws;
    fp.token_ids = token_ids;
    fp.v_offset = v_offset;

    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(pl.grid);
    cfg.blockDim = dim3(kFusedThreads);
    cfg.dynamicSmemBytes = static_cast<size_t>(pl.smem_bytes);
    cfg.stream = stream;
    // Programmatic dependent launch: the kernel may start while the previous kernel in the
    // stream is still running; it executes griddepcontrol.wait before its workspace stores and
    // before it exits (and before its first global read unless overlap is switched on).
    cudaLaunchAttribute fattr[2];
    unsigned na = 0;
    if (use_pdl && allow_pdl) {
        fattr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        fattr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    if (pair) {   // the two CTAs of a pair form a cluster (same TPC)
        fattr[na].id = cudaLaunchAttributeClusterDimension;
        fattr[na].val.clusterDim.x = 2;
        fattr[na].val.clusterDim.y = 1;
        fattr[na].val.clusterDim.z = 1;
        ++na;
    }
    cfg.attrs = fattr;
    cfg.numAttrs = na;
    cudaError_t e = pair ? cudaLaunchKernelEx(&cfg, laser_probe_fused_kernel<true>, tm_h, tm_w, fp)
                         : cudaLaunchKernelEx(&cfg, laser_probe_fused_kernel<false>, tm_h, tm_w, fp);
    if (e != cudaSuccess) return set_cuda_error("launch laser_probe_fused_kernel", e);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return LASER_OK;
}

// The fields of FinalizeParams that describe the fused kernel's workspace for `dims`.
FinalizeParams finalize_params(const DeviceInfo* di, const laser_probe_plan& pl, const laser_probe_dims& dims,
                               bool run_fused, const int32_t* req_offsets) {
    FinalizeParams fz{};
    fz.n_alloc = dims.N; fz.R = dims.R; fz.splits = pl.ws_splits; fz.n_pad = pl.m_tiles * pl.tile_m;
    fz.m_tiles = pl.m_tiles; fz.rows_per_item = pl.tile_m;
    fz.total_tiles = ceil_div(dims.V, pl.tile_n);
    fz.units = units_for(di, pl.cta_pair != 0);
    fz.replan = (run_fused && pl.m_tiles > 1) ? 1 : 0;
    fz.req_offsets = req_offsets;
    fz.wait_flags = nullptr; fz.epoch = 0; fz.a_offset = 0; fz.prob_mode = 0; fz.agg_mode = 0;
    return fz;
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

}  // namespace

// ============================================================================================ ABI
extern "C" {

int laser_tau_params_default(laser_tau_params* out) {
    if (!out) return LASER_E_NULL;
    *out = laser_tau_params{0.95f, 0.04f, 1.0f, 10.0f, 0.88f, 0.97f};
    return LASER_OK;
}

int laser_probe_plan_query(const laser_probe_dims* dims, laser_probe_plan* plan) {
    if (!dims || !plan) return LASER_E_NULL;
    if (!dims_valid(dims)) return LASER_E_DIMS;
    bool ok = false;
    DeviceInfo* di = current_device(&ok);
    make_plan(*dims, (ok && di) ? di->sms : kDefaultSMs, plan);
    return LASER_OK;
}

size_t laser_probe_workspace_bytes(const laser_probe_dims* dims) {
    laser_probe_plan pl;
    if (laser_probe_plan_query(dims, &pl) != LASER_OK) return 0;
    return workspace_bytes_for(pl);
}

int laser_probe_confidence_opt(const void* hidden, const void* W, const int32_t* req_offsets,
                               const float* load, const laser_tau_params* tau_params,
                               float* out_conf, int32_t* out_argmax, uint8_t* out_exit,
                               const laser_probe_dims* dims, void* workspace,
                               size_t workspace_bytes, void* stream_v, float* out_tau_opt,
                               float* out_pmax_opt, const laser_probe_options* options) {
    if (!dims || !tau_params) return LASER_E_NULL;
    if (!dims_valid(dims)) return LASER_E_DIMS;
    if (!params_valid(tau_params)) return LASER_E_PARAMS;
    laser_probe_options opt{LASER_AGG_MEAN, LASER_PROB_MAX, nullptr};
    if (options) opt = *options;
    int rc = options_valid(opt, dims->N);
    if (rc != LASER_OK) return rc;
    const int N = dims->N, R = dims->R;
    if (N == 0 && R == 0) return LASER_OK;
    if (N > 0 && (!hidden || !W || !out_argmax)) return LASER_E_NULL;
    if (R > 0 && (!req_offsets || !load || !out_conf || !out_exit)) return LASER_E_NULL;
    if ((reinterpret_cast<uintptr_t>(hidden) & 15) || (reinterpret_cast<uintptr_t>(W) & 15))
        return LASER_E_ALIGN;

    DeviceInfo* di = nullptr;
    rc = require_b200(&di);
    if (rc != LASER_OK) return rc;
    laser_probe_plan pl;
    make_plan(*dims, di->sms, &pl);
    if (!workspace || workspace_bytes < workspace_bytes_for(pl) ||
        (reinterpret_cast<uintptr_t>(workspace) & 15))
        return LASER_E_WORKSPACE;

    cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
    const bool run_fused = (N > 0 && R > 0);
    const bool prof = g_prof.on && g_prof.created && run_fused && g_prof.calls < kProfRing;
    const int prof_slot = g_prof.calls;
    if (run_fused) {
        if (prof) cudaEventRecord(g_prof.ev[prof_slot][0], stream);
        rc = launch_fused(di, pl, hidden, W, req_offsets, *dims,
                          opt.prob_mode == LASER_PROB_TOKEN ? opt.token_ids : nullptr, 0,
                          static_cast<float4*>(workspace), stream, !prof);
        if (rc != LASER_OK) return rc;
    }

    FinalizeParams fz = finalize_params(di, pl, *dims, run_fused, req_offsets);
    fz.agg_mode = opt.aggregate_mode;
    fz.prob_mode = opt.prob_mode;
    fz.ws = static_cast<const float4*>(workspace);
    fz.row_stride = pl.ws_splits; fz.split_stride = 1;
    fz.load = load;
    fz.out_conf = out_conf; fz.out_argmax = out_argmax; fz.out_exit = out_exit;
    fz.out_tau = out_tau_opt; fz.out_pmax = out_pmax_opt;
    fz.tau = to_dev(tau_params);
    // N == 0 with R > 0: every request is empty -> conf 0, exit 0, tau still defined.  Handled by the
    // same kernel (fz.R = R): req_offsets are all 0, no partials are read.
    if (prof) cudaEventRecord(g_prof.ev[prof_slot][1], stream);
    rc = launch_finalize(fz, stream, run_fused && !prof);
    if (rc != LASER_OK) return rc;
    if (prof) { cudaEventRecord(g_prof.ev[prof_slot][2], stream); g_prof.calls++; }
    return LASER_OK;
}

int laser_probe_confidence_agg(const void* hidden, const void* W, const int32_t* req_offsets,
                               const float* load, const laser_tau_params* tau_params,
                               float* out_conf, int32_t* out_argmax, uint8_t* out_exit,
                               const laser_probe_dims* dims, void* workspace,
                               size_t workspace_bytes, void* stream, float* out_tau_opt,
                               float* out_pmax_opt, int aggregate_mode) {
    const laser_probe_options opt{aggregate_mode, LASER_PROB_MAX, nullptr};
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

// ------------------------------------------------------------------------------ vocabulary-parallel
int laser_probe_partial(const void* hidden, const void* W_shard, const int32_t* req_offsets,
                        const int32_t* token_ids_opt, const laser_probe_dims* dims, int32_t v_offset,
                        laser_row_stats* out_stats, const laser_probe_peers* peers_opt,
                        void* workspace, size_t workspace_bytes, void* stream_v) {
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
    const int N = dims->N, R = dims->R;
    if (N > 0 && (!hidden || !W_shard)) return LASER_E_NULL;
    if (R > 0 && !req_offsets) return LASER_E_NULL;
    if ((reinterpret_cast<uintptr_t>(hidden) & 15) || (reinterpret_cast<uintptr_t>(W_shard) & 15) ||
        (reinterpret_cast<uintptr_t>(out_stats) & 15))
        return LASER_E_ALIGN;
    DeviceInfo* di = nullptr;
    int rc = require_b200(&di);
    if (rc != LASER_OK) return rc;
    laser_probe_plan pl;
    make_plan(*dims, di->sms, &pl);
    if (!workspace || workspace_bytes < workspace_bytes_for(pl) ||
        (reinterpret_cast<uintptr_t>(workspace) & 15))
        return LASER_E_WORKSPACE;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
    const bool run_fused = (N > 0 && R > 0);
    if (run_fused) {
        rc = launch_fused(di, pl, hidden, W_shard, req_offsets, *dims, token_ids_opt, v_offset,
                          static_cast<float4*>(workspace), stream, true);
        if (rc != LASER_OK) return rc;
    }
    if (N > 0) {
        ReduceParams rq{};
        rq.f = finalize_params(di, pl, *dims, run_fused, req_offsets);
        rq.f.R = run_fused ? R : 0;            // R == 0: every row is padding -> neutral records
        rq.f.ws = static_cast<const float4*>(workspace);
        rq.f.row_stride = pl.ws_splits; rq.f.split_stride = 1;
        rq.f.a_offset = v_offset;
        rq.out_stats = reinterpret_cast<float4*>(out_stats);
        rq.rank = peers_opt ? peers_opt->rank : 0;
        rq.world = peers_opt ? peers_opt->world : 0;
        for (int g = 0; g < rq.world; ++g) rq.peer_stats[g] = reinterpret_cast<float4*>(peers_opt->peer_stats[g]);
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
        SignalParams sg{};
        sg.rank = peers_opt->rank; sg.world = peers_opt->world; sg.epoch = peers_opt->epoch;
        for (int g = 0; g < sg.world; ++g) sg.peer_flags[g] = peers_opt->peer_flags[g];
        laser_probe_signal_kernel<<<1, 32, 0, stream>>>(sg);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return set_cuda_error("launch laser_probe_signal_kernel", e);
        g_launches.fetch_add(1, std::memory_order_relaxed);
    }
    return LASER_OK;
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
    laser_probe_options opt{LASER_AGG_MEAN, LASER_PROB_MAX, nullptr};
    if (options) opt = *options;
    if (opt.aggregate_mode < LASER_AGG_MEAN || opt.aggregate_mode > LASER_AGG_MIN ||
        opt.prob_mode < LASER_PROB_MAX || opt.prob_mode > LASER_PROB_TOKEN)
        return LASER_E_MODE;
    const int N = dims->N, R = dims->R;
    if (N == 0 && R == 0) return LASER_OK;
    if (N > 0 && (!stats || !out_argmax)) return LASER_E_NULL;
    if (R > 0 && (!req_offsets || !load || !out_conf || !out_exit)) return LASER_E_NULL;
    if (reinterpret_cast<uintptr_t>(stats) & 15) return LASER_E_ALIGN;
    DeviceInfo* di = nullptr;
    int rc = require_b200(&di);
    if (rc != LASER_OK) return rc;
    FinalizeParams fz{};
    fz.n_alloc = N; fz.R = R; fz.splits = G; fz.n_pad = N;
    fz.m_tiles = 1; fz.rows_per_item = kTileM; fz.total_tiles = 1; fz.units = 1; fz.replan = 0;
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
    return launch_finalize(fz, static_cast<cudaStream_t>(stream_v), false);
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
        e = cudaMemcpyAsync(base + st.hidden, h_hidden, static_cast<size_t>(n_copy) * dims->d * 2,
                            cudaMemcpyHostToDevice, stream);
        if (e != cudaSuccess) return set_cuda_error("H2D hidden", e);
    }
    // Zero-copy for the small tensors: when req_offsets, load and the three outputs all live in
    // pinned, device-mapped host memory (cudaHostAlloc / cudaHostRegister / torch pin_memory), the
    // finalize kernel reads and writes them over PCIe directly — the reads overlap the fused kernel
    // (they precede griddepcontrol.wait) — and the call issues one copy (hidden) instead of six.
    auto mapped = [](const void* h) -> void* {
        if (!h) return nullptr;
        cudaPointerAttributes a;
        if (cudaPointerGetAttributes(&a, h) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
        return a.type == cudaMemoryTypeHost ? a.devicePointer : nullptr;
    };
    void* m_off = R > 0 ? mapped(h_req_offsets) : nullptr;
    void* m_load = R > 0 ? mapped(h_load) : nullptr;
    void* m_conf = R > 0 ? mapped(h_out_conf) : nullptr;
    void* m_exit = R > 0 ? mapped(h_out_exit) : nullptr;
    void* m_arg = N > 0 ? mapped(h_out_argmax) : nullptr;
    const bool zero_copy = (R == 0 || (m_off && m_load && m_conf && m_exit)) && (N == 0 || m_arg);
    if (zero_copy) {
        int rc = laser_probe_confidence(base + st.hidden, W, static_cast<int32_t*>(m_off),
                                        static_cast<float*>(m_load), tau_params,
                                        static_cast<float*>(m_conf), static_cast<int32_t*>(m_arg),
                                        static_cast<uint8_t*>(m_exit), dims, workspace, workspace_bytes,
                                        stream_v, nullptr, nullptr);
        if (rc != LASER_OK) return rc;
    } else {
        if (R > 0) {
            e = cudaMemcpyAsync(base + st.offsets, h_req_offsets, static_cast<size_t>(R + 1) * 4,
                                cudaMemcpyHostToDevice, stream);
            if (e != cudaSuccess) return set_cuda_error("H2D req_offsets", e);
            e = cudaMemcpyAsync(base + st.load, h_load, static_cast<size_t>(R) * 4, cudaMemcpyHostToDevice, stream);
            if (e != cudaSuccess) return set_cuda_error("H2D load", e);
        }
        int rc = laser_probe_confidence(base + st.hidden, W, reinterpret_cast<int32_t*>(base + st.offsets),
                                        reinterpret_cast<float*>(base + st.load), tau_params,
                                        reinterpret_cast<float*>(base + st.conf),
                                        reinterpret_cast<int32_t*>(base + st.argmax), base + st.exit_, dims,
                                        workspace, workspace_bytes, stream_v, nullptr, nullptr);
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
    return LASER_OK;
}

int laser_probe_confidence_host(const void* h_hidden, const void* W, const int32_t* h_req_offsets,
                                const float* h_load, const laser_tau_params* tau_params,
                                float* h_out_conf, int32_t* h_out_argmax, uint8_t* h_out_exit,
                                const laser_probe_dims* dims, void* workspace,
                                size_t workspace_bytes, void* d_staging, size_t staging_bytes,
                                void* stream_v) {
    int rc = laser_probe_confidence_host_async(h_hidden, W, h_req_offsets, h_load, tau_params, h_out_conf,
                                               h_out_argmax, h_out_exit, dims, workspace, workspace_bytes,
                                               d_staging, staging_bytes, stream_v);
    if (rc != LASER_OK) return rc;
    if (dims->N == 0 && dims->R == 0) return LASER_OK;
    cudaError_t e = cudaStreamSynchronize(static_cast<cudaStream_t>(stream_v));
    if (e != cudaSuccess) return set_cuda_error("cudaStreamSynchronize", e);
    return LASER_OK;
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
    *out = laser_budget_params{10.f, 2.f, 0.6f, 1.5f, 50.f, 275.f, 10.f};
    return LASER_OK;
}

int laser_allocate_budget(const int32_t* prompt_tokens, const float* L, int32_t R,
                          const laser_budget_params* q, int32_t* out_budget) {
    if (!q || (R > 0 && (!prompt_tokens || !L || !out_budget))) return LASER_E_NULL;
    if (R < 0) return LASER_E_DIMS;
    if (!(q->p_max > q->p_min) || !(q->f_max >= q->f_min) || !(q->l_target > 0.f)) return LASER_E_PARAMS;
    for (int32_t r = 0; r < R; ++r) {
        // Eq. 7: difficulty factor from the prompt length, clipped to [f_min, f_max]
        double f_diff = q->f_min + (static_cast<double>(prompt_tokens[r]) - q->p_min) /
                                       (static_cast<double>(q->p_max) - q->p_min) *
                                       (static_cast<double>(q->f_max) - q->f_min);
        f_diff = f_diff < q->f_min ? q->f_min : (f_diff > q->f_max ? q->f_max : f_diff);
        // Eq. 8: load factor min(1, L_target / max(1, L(t)))
        const double den = L[r] > 1.f ? L[r] : 1.0;
        double f_load = q->l_target / den;
        f_load = f_load < 1.0 ? f_load : 1.0;
        // Eq. 6
        double b = std::floor(static_cast<double>(q->b_base) * f_diff * f_load);
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
        case LASER_E_MODE: return "unknown aggregate mode";
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

int laser_probe_set_mode(int mode) {
    if (mode < LASER_MODE_AUTO || mode > LASER_MODE_PAIR) return LASER_E_MODE;
    g_force_mode.store(mode, std::memory_order_relaxed);
    return LASER_OK;
}

int laser_probe_set_overlap(int enable) {
    g_overlap.store(enable ? 1 : 0, std::memory_order_relaxed);
    return LASER_OK;
}

const char* laser_last_error(void) { return g_last_error.c_str(); }

uint64_t laser_kernel_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

int laser_shutdown(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    g_maps.clear();
    return LASER_OK;
}

}  // extern "C"
