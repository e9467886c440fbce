// xy_api.cu -- the C ABI of include/xy.h: host-side bookkeeping and kernel launches.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -shared -Xcompiler -fPIC
#include "../../include/xy.h"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <utility>
#include <vector>

#include "xy_kernels.cuh"
#include "xy_resident.cuh"

using namespace xyk;

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) return fail(XY_ERR_CUDA, "%s failed: %s", #call, cudaGetErrorString(e_)); \
    } while (0)

constexpr int kMaxDevices = 64;
size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }
bool shape_ok(int L, int R) { return L >= 8 && L % 8 == 0 && L <= 1024 && R >= 1 && R <= 65535; }
size_t max_tiles(int L) { return (size_t)(L / 2) * (size_t)(L / 2); }   // tiles_ok: TY >= 2 and TZ >= 2

struct WsLayout {
    size_t obs_rank, obs_slot, partials, partials6, obs6, dctr, betas, beta_of_slot, beta32, slot_at_rank, met_acc, pt_acc, exact, near_ctl, res_sync, res_xchg, near_queue, stage, total;
    unsigned int near_cap;
};
WsLayout ws_layout(int L, int R) {
    WsLayout w;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
    w.obs_rank = take((size_t)R * 5 * 8);
    w.obs_slot = take((size_t)R * 5 * 8);
    w.partials = take((size_t)R * max_tiles(L) * 3 * 8);
    w.partials6 = take((size_t)R * max_tiles(L) * 6 * 8);
    w.obs6 = take((size_t)R * 6 * 8);
    w.dctr = take(sizeof(DeviceCounters));
    w.betas = take((size_t)R * 8);
    w.beta_of_slot = take((size_t)R * 8);
    w.beta32 = take((size_t)R * 4);
    w.slot_at_rank = take((size_t)R * 4);
    w.met_acc = take((size_t)R * 8);
    w.pt_acc = take((size_t)R * 8);
    w.exact = take(8);
    w.near_ctl = take(16);                           // near_count, done_ticket, overflow_flag
    w.res_sync = take(16);                           // resident kernel: grid barrier counter, error flag
    w.res_xchg = take((size_t)2 * (R <= kResMaxR ? R : 0) * kResMaxC * 6 * 8);   // resident kernel: published partial sums
    // capacity of the close-decision queue: 2e-3 of one colour pass (expected load at beta ~ 0.45 is 4e-5)
    const size_t pass_sites = (size_t)R * L * L * L / 2;
    size_t cap = (size_t)((double)pass_sites * 2e-3);
    if (cap < 4096) cap = 4096;
    w.near_cap = (unsigned int)cap;
    w.near_queue = take(cap * 16);
    w.stage = take((size_t)L * L * L * 4);
    w.total = o;
    return w;
}

// resident path (xy_resident.cuh): slots per CTA or CTAs per slot, launch shape.  Dynamic + static shared memory of a
// block may not exceed the 227 KB opt-in limit: 1 KB is left for the kernel's static variables.
constexpr size_t kResidentSmemMax = 226 * 1024;
struct ResidentPlan { bool ok = false; int G = 1, C = 1, tps = 0, threads = 0, grid = 0; size_t smem = 0; };

}  // namespace

struct xy_ctx {
    int L = 0, R = 0;
    size_t N = 0, half_n = 0;
    uint64_t seed = 0;
    std::vector<double> betas;
    PhiloxKeys keys;
    uint32_t n_met = 0, n_or = 0, n_pt = 0;
    // device
    int device = -1;                           // the CUDA device of the attached buffers and stream (xy_attach)
    int sm_count = 148;                        // its multiprocessors (xy_attach)
    bool attached = false;
    float* d_state = nullptr; bool own_state = false;
    char* d_ws = nullptr; bool own_ws = false;
    cudaStream_t stream = nullptr; bool own_stream = false;
    WsLayout ws;
    float* d_trace = nullptr;
    // options
    int TY = 0, TZ = 0, TY_met = 0, TZ_met = 0, trace = 0, fused = 1, generic = 0, or_per_mcs = 1, use_graph = 1, resident = 1, slot_chunk = 0;
    bool res_planned = false, res_used = false;   // resident path: plan cached; a launch is in flight whose error flag must be read
    ResidentPlan res_plan;
    bool slot_valid = false;                   // obs_slot holds the observables of the current spins (resident kernel)
    // CUDA graph of one Monte Carlo step in device-counter mode (xy_mcs), rebuilt when graph_key changes
    cudaGraphExec_t graph_exec = nullptr;
    uint64_t graph_key = 0, graph_launches = 0;
    bool device_counters = false;              // true while a step is being enqueued for capture
    // cache state
    bool partials_valid = false, rank_valid = false;
    uint64_t launches = 0;
    // XY_OPT_PROFILE: one CUDA-event pair around every launch, resolved by xy_get_kernel_times
    int profile = 0;
    struct Span { cudaEvent_t a, b; int cls; };
    std::vector<Span> spans;
    std::vector<cudaEvent_t> free_events;
    double k_ms[XY_NUM_KERNEL_CLASSES] = {};
    uint64_t k_n[XY_NUM_KERNEL_CLASSES] = {};

    float* colour(int c) const { return d_state + (size_t)c * R * half_n; }
    template <class T> T* ws_ptr(size_t off) const { return reinterpret_cast<T*>(d_ws + off); }
};

namespace {

// Brackets one kernel launch with a pair of events on the context's stream when profiling is on.
struct LaunchSpan {
    xy_ctx* c; int cls; cudaEvent_t a = nullptr, b = nullptr;
    static cudaEvent_t take(xy_ctx* c) {
        cudaEvent_t e = nullptr;
        if (!c->free_events.empty()) { e = c->free_events.back(); c->free_events.pop_back(); }
        else if (cudaEventCreate(&e) != cudaSuccess) e = nullptr;
        return e;
    }
    LaunchSpan(xy_ctx* ctx, int k) : c(ctx), cls(k) {
        ++c->launches;
        if (!c->profile) return;
        a = take(c); b = take(c);
        if (a) cudaEventRecord(a, c->stream);
    }
    ~LaunchSpan() {
        if (!c->profile || !a || !b) return;
        cudaEventRecord(b, c->stream);
        c->spans.push_back({a, b, cls});
    }
};

// Multiprocessors of the device the tiles are chosen for: the current device if there is one (a query only -- no
// context is created, nothing is allocated), else a full B200.  The tile models below count block slots in units of
// this number instead of assuming 148.
constexpr int kB200Sms = 148;
int current_sm_count() {
    int n_dev = 0, dev = 0, sms = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1) { cudaGetLastError(); return kB200Sms; }
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
        cudaGetLastError();
        return kB200Sms;
    }
    return sms;
}

void default_tiles_z(int L, int R, int TY, int& TZ, int sms);

void default_tiles(int L, int R, int& TY, int& TZ, int sms = 0) {
    if (sms <= 0) sms = current_sm_count();
    const int W4 = L / 8;
    TY = 2;                                        // L up to 1024: TY * L/8 must stay within 11 compute warps
    for (int t = 2; t <= L; ++t)
        if (L % t == 0 && t * W4 <= 320) TY = t;
    default_tiles_z(L, R, TY, TZ, sms);
}

// March length for tile rows TY on a device of `sms` multiprocessors.
void default_tiles_z(int L, int R, int TY, int& TZ, int sms) {
    // A block costs TZ + 2 steps (two of them only stage) plus the latency of its first copies (about
    // 1.5 step-times), and 2 blocks fit an SM.  With w = blocks / (2 * sms) "waves" the pass takes about
    // (max(w, 1/2) + 0.3) * (TZ + 3.5) step-times: blocks end at different times, so a fraction of a wave is lost at the
    // end, not a whole one, and an SM that holds one block instead of two runs it faster.  Take the divisor of L that
    // minimises it.  Fitted to the measured march-length sweeps at L = 64, 128, 160 (profiles/r2_experiments.md).
    TZ = L;
    double best = 1e300;
    for (int t = L; t >= 2; --t) {
        if (L % t) continue;
        const double w = (double)((long)R * (L / TY) * (L / t)) / (2.0 * sms);
        const double cost = (std::fmax(w, 0.5) + 0.3) * (t + 3.5);
        if (cost < best * 0.999) { best = cost; TZ = t; }
    }
}

bool tiles_ok(int L, int TY, int TZ) {
    return TY >= 2 && TZ >= 2 && L % TY == 0 && L % TZ == 0 && TY * (L / 8) <= 352 &&   // 11 compute warps + the auxiliary warp
           sweep_smem_bytes_max(L, TY) <= 200 * 1024;
}

// Launches one kernel of the step's chain.  With XY_PDL the launch carries the programmatic-stream-serialization
// attribute (xy_device.cuh): its blocks may become resident during the tail of the previous kernel on the stream and
// wait there (grid_dependency_wait) until that kernel has completed.  Profiling puts event records between the
// launches, which serialises them the ordinary way.
template <class... KArgs, class... Args>
cudaError_t launch_chained(bool pdl, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args&&... args) {
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

// Where it pays: the saving is a few microseconds per kernel boundary, so +1 ... +5 % per step for passes of up to ~7
// blocks per multiprocessor (L = 64 ... 128 x 34 replicas, L = 160 x 13; profiles/r3_experiments.md), while at
// L = 160 x 64 (9-11 blocks per multiprocessor and pass) the step was 0.15 % SLOWER with it, repeatably.  Hence the bound.
bool chain_pdl(const xy_ctx* c) {
    return XY_PDL != 0 && (long)c->R * (c->L / c->TY) * (c->L / c->TZ) <= 8L * c->sm_count;
}

template <int MODE, bool TRACE, bool FUSED, bool EXACT_INLINE, int W4C, int TYC>
int launch_sweep_impl(xy_ctx* c, const SweepParams& P) {
    // Two instantiations per variant: with and without the grid-dependency instructions (the test hook and the
    // large-|beta| variant only without).  The dynamic-shared-memory opt-in is a per-device attribute of each: one flag
    // per device, set outside any stream capture (xy_mcs launches its first step eagerly).
    constexpr bool CAN_PDL = XY_PDL != 0 && !TRACE && !EXACT_INLINE;
    auto plain = sweep_kernel<MODE, TRACE, FUSED, EXACT_INLINE, W4C, TYC, false>;
    auto chained = sweep_kernel<MODE, TRACE, FUSED, EXACT_INLINE, W4C, TYC, CAN_PDL>;
    static std::atomic<bool> attr_set[kMaxDevices];
    if (!attr_set[c->device].load(std::memory_order_acquire)) {
        CK(cudaFuncSetAttribute(plain, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        if (CAN_PDL) CK(cudaFuncSetAttribute(chained, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        attr_set[c->device].store(true, std::memory_order_release);
    }
    const size_t smem = sweep_smem_bytes(P.L, P.TY, W4C != 0 && (W4C * TYC / 2) % 32 == 0);   // the kernel's UNI mapping
    const int threads = (P.nItems + 31) / 32 * 32 + 32;          // compute warps + the auxiliary warp
    dim3 grid(P.nTY * P.nTZ, P.n_slots);
    const bool pdl = CAN_PDL && chain_pdl(c);
    {
        LaunchSpan span(c, MODE == MODE_MET ? XY_K_METROPOLIS : MODE == MODE_OR ? XY_K_OVERRELAX : XY_K_MEASURE);   // MODE_STIFF counts as measure
        CK(launch_chained(pdl, pdl ? chained : plain, grid, dim3(threads), smem, c->stream, P));
    }
    return XY_OK;
}

// Tile geometry as compile-time constants for the lattice sizes of the paper's workloads
// (L = 32, 64, 80, 96, 128, 160 with their default tiles; at L = 80 no tile has warps of uniform x parity: geometry only); everything else takes the run-time variant of
// the same kernel.  The test hook and the large-|beta| variant are always run-time geometry.
template <int MODE, bool TRACE, bool FUSED, bool EXACT_INLINE = false>
int launch_sweep(xy_ctx* c, const SweepParams& P) {
    if (!TRACE && !EXACT_INLINE && !c->generic) {
        if (MODE == MODE_MET && P.W4 == 20 && P.TY == 32) return launch_sweep_impl<MODE_MET, false, false, false, 20, 32>(c, P);
        if (P.W4 == 20 && P.TY == 16) return launch_sweep_impl<MODE, false, FUSED, false, 20, 16>(c, P);
        if (P.W4 == 16 && P.TY == 16) return launch_sweep_impl<MODE, false, FUSED, false, 16, 16>(c, P);
        if (P.W4 == 12 && P.TY == 16) return launch_sweep_impl<MODE, false, FUSED, false, 12, 16>(c, P);
        if (P.W4 == 10 && P.TY == 16) return launch_sweep_impl<MODE, false, FUSED, false, 10, 16>(c, P);
        if (P.W4 == 8 && P.TY == 32) return launch_sweep_impl<MODE, false, FUSED, false, 8, 32>(c, P);
        if (P.W4 == 4 && P.TY == 32) return launch_sweep_impl<MODE, false, FUSED, false, 4, 32>(c, P);
    }
    return launch_sweep_impl<MODE, TRACE, FUSED, EXACT_INLINE, 0, 0>(c, P);
}

// True when so many Metropolis decisions would fall inside the fp64 window (|beta| large) that the
// close-decision queue could overflow: the sweep then re-evaluates them in the loop instead.
bool need_inline_exact(const xy_ctx* c) {
    double bmax = 0.0;
    for (double b : c->betas) bmax = std::fmax(bmax, std::fabs((double)(float)b));
    const double window = bmax * (double)kWindowPerBeta + (double)kWindowAbs;
    const double pass_sites = (double)c->R * (double)c->N / 2.0;
    return (2.0 * window + 6e-8) * pass_sites > (double)c->ws.near_cap / 8.0;
}

SweepParams base_params(xy_ctx* c, int colour) {
    SweepParams P;
    memset(&P, 0, sizeof(P));
    P.own = c->colour(colour);
    P.other = c->colour(1 - colour);
    P.L = c->L; P.W = c->L / 2; P.W4 = c->L / 8;
    P.TY = c->TY; P.TZ = c->TZ; P.nTY = c->L / c->TY; P.nTZ = c->L / c->TZ;          // xy_metropolis_sweep may override (TY_met)
    P.colour = colour;
    P.slot0 = 0; P.n_slots = c->R;                   // all slots; the chunked schedule of xy_mcs narrows them
    P.nItems = P.TY * P.W4;
    P.half_n = (unsigned int)c->half_n;
    P.keys = c->keys;
    P.beta32_of_slot = c->ws_ptr<float>(c->ws.beta32);
    P.met_acc = c->ws_ptr<unsigned long long>(c->ws.met_acc);
    P.exact_count = c->ws_ptr<unsigned long long>(c->ws.exact);
    P.partials = c->ws_ptr<double>(c->ws.partials);
    P.near_queue = c->ws_ptr<uint4>(c->ws.near_queue);
    P.near_count = c->ws_ptr<unsigned int>(c->ws.near_ctl);
    P.near_cap = c->ws.near_cap;
    P.d_counters = c->device_counters ? c->ws_ptr<uint32_t>(c->ws.dctr) : nullptr;
    return P;
}

// Makes the context's device current for the duration of one entry point and restores the caller's.
struct DeviceScope {
    int prev = -1; bool switched = false;
    int enter(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) return fail(XY_ERR_CUDA, "cudaGetDevice failed");
        if (prev != dev) {
            if (cudaSetDevice(dev) != cudaSuccess) return fail(XY_ERR_CUDA, "cudaSetDevice(%d) failed", dev);
            switched = true;
        }
        return XY_OK;
    }
    ~DeviceScope() { if (switched) cudaSetDevice(prev); }
};

int need(xy_ctx* c) {
    if (!c) return fail(XY_ERR_INVALID_ARG, "NULL context");
    if (!c->attached) return fail(XY_ERR_NOT_ATTACHED, "context has no device buffers: call xy_attach first");
    return XY_OK;
}
// First statement of every entry point that touches the device: validates the context and switches to its device.
#define ENTER(c)                                   \
    if (int rc_ = need(c)) return rc_;             \
    DeviceScope scope_;                            \
    if (int rc_ = scope_.enter((c)->device)) return rc_

int upload_labels(xy_ctx* c, const int* perm) {
    const int R = c->R;
    std::vector<double> bos(R);
    std::vector<float> b32(R);
    std::vector<int> sar(R);
    for (int k = 0; k < R; ++k) { sar[k] = perm ? perm[k] : k; bos[sar[k]] = c->betas[k]; b32[sar[k]] = (float)c->betas[k]; }
    CK(cudaMemcpyAsync(c->ws_ptr<double>(c->ws.betas), c->betas.data(), R * 8, cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->ws_ptr<double>(c->ws.beta_of_slot), bos.data(), R * 8, cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->ws_ptr<float>(c->ws.beta32), b32.data(), R * 4, cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->ws_ptr<int>(c->ws.slot_at_rank), sar.data(), R * 4, cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));     // the host vectors die here
    c->rank_valid = false;
    return XY_OK;
}

// After a stream synchronise: fail loudly if a colour pass ever produced more close decisions than
// the queue holds (then some decisions kept their fp32 value; see need_inline_exact).
int check_near_overflow(xy_ctx* c) {
    unsigned int flag = 0;
    CK(cudaMemcpyAsync(&flag, c->ws_ptr<unsigned int>(c->ws.near_ctl) + 2, 4, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    if (flag) return fail(XY_ERR_CUDA, "Metropolis close-decision queue overflowed (capacity %u): results are not exact", c->ws.near_cap);
    if (c->res_used) {                         // the resident kernel's grid barrier timed out (its CTAs were not co-resident)
        unsigned int err = 0;
        CK(cudaMemcpyAsync(&err, c->ws_ptr<unsigned int>(c->ws.res_sync) + 1, 4, cudaMemcpyDeviceToHost, c->stream));
        CK(cudaStreamSynchronize(c->stream));
        if (err) return fail(XY_ERR_CUDA, "resident Monte Carlo kernel aborted at its grid barrier: results are invalid");
    }
    return XY_OK;
}

int grid_for(size_t n_items, int threads) {
    size_t b = (n_items + threads - 1) / threads;
    static const size_t cap = (size_t)current_sm_count() * 16;      // grid-stride kernels: 16 blocks per multiprocessor at most
    return (int)(b < 1 ? 1 : (b > cap ? cap : b));
}

int run_measure(xy_ctx* c, double* d_series_row) {
    if (!c->partials_valid && c->slot_valid) {           // the resident kernel left the by-slot observables of these spins
        if (!c->rank_valid) {
            LaunchSpan span(c, XY_K_FINALIZE);
            gather_rank_kernel<<<(5 * c->R + 127) / 128, 128, 0, c->stream>>>(c->ws_ptr<double>(c->ws.obs_slot), c->ws_ptr<int>(c->ws.slot_at_rank),
                                                                              c->R, c->ws_ptr<double>(c->ws.obs_rank));
            CK(cudaGetLastError());
            c->rank_valid = true;
        }
        return XY_OK;
    }
    if (!c->partials_valid) {
        SweepParams P = base_params(c, 1);     // own = white, staged = black
        int rc = launch_sweep<MODE_MEASURE, false, false>(c, P);
        if (rc) return rc;
        c->partials_valid = true;
        c->rank_valid = false;
    }
    if (!c->rank_valid || d_series_row) {
        const int n_tiles = (c->L / c->TY) * (c->L / c->TZ);
        {
            LaunchSpan span(c, XY_K_FINALIZE);
            measure_finalize_kernel<<<(c->R + 3) / 4, 128, 0, c->stream>>>(c->ws_ptr<double>(c->ws.partials), n_tiles, c->R,
                                                                 c->ws_ptr<int>(c->ws.slot_at_rank),
                                                                 c->ws_ptr<double>(c->ws.obs_rank),
                                                                 c->ws_ptr<double>(c->ws.obs_slot), d_series_row);
        }
        CK(cudaGetLastError());
        c->rank_valid = true;
    }
    return XY_OK;
}


// ---- resident path (xy_resident.cuh): one persistent launch for n whole steps of a small lattice ------------------
template <int L, int C>
int resident_launch(xy_ctx* c, const ResidentPlan& pl, const ResidentParams& P, bool query_only, int* max_clusters) {
    constexpr bool CLUSTER = C > 1;
    auto kern = resident_mcs_kernel<L, C>;
    static std::atomic<bool> attr_set[kMaxDevices];
    if (!attr_set[c->device].load(std::memory_order_acquire)) {
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kResidentSmemMax));
        attr_set[c->device].store(true, std::memory_order_release);
    }
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(pl.grid); cfg.blockDim = dim3(pl.threads); cfg.dynamicSmemBytes = pl.smem; cfg.stream = c->stream;
    cudaLaunchAttribute at[2];
    int na = 0;
    if (CLUSTER) { at[na].id = cudaLaunchAttributeClusterDimension; at[na].val.clusterDim.x = C; at[na].val.clusterDim.y = 1; at[na].val.clusterDim.z = 1; ++na; }
    cfg.attrs = at; cfg.numAttrs = na;
    if (query_only) {                          // how many clusters (CTAs for C = 1) of this shape can be resident at once?
        if (CLUSTER) { CK(cudaOccupancyMaxActiveClusters(max_clusters, kern, &cfg)); }
        else {
            int per_sm = 0, dev_sms = 0;
            CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, pl.threads, pl.smem));
            CK(cudaDeviceGetAttribute(&dev_sms, cudaDevAttrMultiProcessorCount, c->device));
            *max_clusters = per_sm * dev_sms;
        }
        return XY_OK;
    }
    // the CTAs wait on one another once per step: co-residency is guaranteed by a cooperative launch
    at[na].id = cudaLaunchAttributeCooperative; at[na].val.cooperative = 1; ++na;
    cfg.numAttrs = na;
    // res_sync[1], the kernel's "aborted" flag, is zeroed by xy_attach only: like the close-decision overflow flag it stays
    // set until the context is attached again, so a second xy_mcs enqueued before any synchronising call cannot wipe it
    if (pl.grid > 1) CK(cudaMemsetAsync(c->ws_ptr<char>(c->ws.res_xchg), 0, (size_t)2 * c->R * kResMaxC * 6 * 8, c->stream));   // step tags start at 1
    {
        LaunchSpan span(c, XY_K_RESIDENT);
        CK(cudaLaunchKernelEx(&cfg, kern, P));
    }
    return XY_OK;
}

// The (L, C) pairs with a kernel: every slab with its two halo planes must fit in one block's shared memory.
int resident_dispatch(xy_ctx* c, const ResidentPlan& pl, const ResidentParams& P, bool query_only, int* max_clusters) {
#define XY_RES_CASE(LL, CC) if (c->L == LL && pl.C == CC) return resident_launch<LL, CC>(c, pl, P, query_only, max_clusters)
    XY_RES_CASE(8, 1);
    XY_RES_CASE(16, 1); XY_RES_CASE(16, 2); XY_RES_CASE(16, 4); XY_RES_CASE(16, 8);
    XY_RES_CASE(24, 1); XY_RES_CASE(24, 2); XY_RES_CASE(24, 4); XY_RES_CASE(24, 8);
    XY_RES_CASE(32, 2); XY_RES_CASE(32, 4); XY_RES_CASE(32, 8);
    XY_RES_CASE(40, 8);
    XY_RES_CASE(48, 8);
#undef XY_RES_CASE
    return fail(XY_ERR_INVALID_ARG, "no resident kernel for L=%d with %d thread blocks per slot", c->L, pl.C);
}
bool resident_has_kernel(int L, int C) {
    switch (L) {
        case 8: return C == 1;
        case 16: case 24: return C == 1 || C == 2 || C == 4 || C == 8;
        case 32: return C == 2 || C == 4 || C == 8;
        case 40: case 48: return C == 8;
        default: return false;
    }
}

// Chooses slots per CTA (tiny lattices) or CTAs per slot (a cluster), such that everything fits in shared memory and ALL
// CTAs are resident at once (they meet once per step).  Cached per context.
const ResidentPlan& resident_plan(xy_ctx* c) {
    if (c->res_planned) return c->res_plan;
    c->res_planned = true;
    ResidentPlan& best = c->res_plan;
    const int L = c->L, R = c->R;
    if (R > kResMaxR) return best;
    ResidentParams dummy;
    memset(&dummy, 0, sizeof(dummy));
    const int pi = resident_plane_items(L), maxt = resident_max_threads(L);
    for (int C = kResMaxC; C >= 1; C >>= 1) {              // the largest co-resident cluster per slot: most SMs at work
        if (!resident_has_kernel(L, C)) continue;
        ResidentPlan pl;
        pl.C = C;
        pl.G = C == 1 ? (R + 131) / 132 : 1;               // tiny lattices, many slots: several slots per CTA
        int unit = pi;                                     // threads per slot: whole planes; whole warps too if slots share a block
        if (pl.G > 1) while (unit % 32) unit += pi;
        const int items = (L / C) * pi;
        int tps = (items + unit - 1) / unit * unit;
        if (tps > maxt / pl.G) tps = maxt / pl.G / unit * unit;
        if (tps < unit) continue;
        pl.tps = tps;
        pl.threads = (tps * pl.G + 31) / 32 * 32;
        pl.grid = C == 1 ? (R + pl.G - 1) / pl.G : R * C;
        pl.smem = resident_smem_bytes(L, R, pl.G, C);
        if (pl.smem > kResidentSmemMax) continue;
        int cap = 0;
        if (resident_dispatch(c, pl, dummy, true, &cap) != XY_OK) { cudaGetLastError(); continue; }
        if (cap >= (C == 1 ? pl.grid : R)) { pl.ok = true; best = pl; break; }    // cap counts clusters (CTAs for C = 1)
        fail(XY_OK, "resident plan: L=%d R=%d needs %d clusters of %d thread blocks, %d can be resident", L, R, C == 1 ? pl.grid : R, C, cap);
    }
    return best;
}

int resident_mcs(xy_ctx* c, const ResidentPlan& pl, int n_mcs, double* d_series) {
    ResidentParams P;
    memset(&P, 0, sizeof(P));
    P.black = c->colour(0); P.white = c->colour(1);
    P.R = c->R; P.n_mcs = n_mcs; P.or_per_mcs = c->or_per_mcs; P.G = pl.G; P.tps = pl.tps;
    P.n_met0 = c->n_met; P.n_pt0 = c->n_pt; P.keys = c->keys;
    P.betas = c->ws_ptr<double>(c->ws.betas);
    P.beta_of_slot = c->ws_ptr<double>(c->ws.beta_of_slot); P.beta32_of_slot = c->ws_ptr<float>(c->ws.beta32);
    P.slot_at_rank = c->ws_ptr<int>(c->ws.slot_at_rank);
    P.met_acc = c->ws_ptr<unsigned long long>(c->ws.met_acc); P.pt_acc = c->ws_ptr<unsigned long long>(c->ws.pt_acc);
    P.exact_count = c->ws_ptr<unsigned long long>(c->ws.exact);
    P.obs_rank = c->ws_ptr<double>(c->ws.obs_rank); P.obs_slot = c->ws_ptr<double>(c->ws.obs_slot);
    P.series = d_series;
    P.xchg = c->ws_ptr<unsigned long long>(c->ws.res_xchg);
    P.sync = c->ws_ptr<unsigned int>(c->ws.res_sync);
    if (const int rc = resident_dispatch(c, pl, P, false, nullptr)) return rc;
    c->n_met += (uint32_t)n_mcs; c->n_or += (uint32_t)n_mcs * (uint32_t)c->or_per_mcs; c->n_pt += (uint32_t)n_mcs;
    c->partials_valid = false; c->slot_valid = true;       // by-slot observables of the final spins are on the device
    c->rank_valid = false;                                 // the by-rank rows belong to the labelling before the last exchange
    c->res_used = true;
    return XY_OK;
}

}  // namespace

extern "C" {

const char* xy_last_error(void) { return g_err; }

xy_ctx* xy_create(int L, int R, const double* betas, uint64_t seed) {
    if (!shape_ok(L, R)) { fail(XY_ERR_INVALID_ARG, "xy_create: need L %% 8 == 0, 8 <= L <= 1024, 1 <= R <= 65535 (got L=%d R=%d)", L, R); return nullptr; }
    if (!betas) { fail(XY_ERR_INVALID_ARG, "xy_create: betas is NULL"); return nullptr; }
    for (int k = 0; k < R; ++k)
        if (!std::isfinite(betas[k])) { fail(XY_ERR_INVALID_ARG, "xy_create: betas[%d] is not finite", k); return nullptr; }
    xy_ctx* c = new xy_ctx;
    c->L = L; c->R = R; c->N = (size_t)L * L * L; c->half_n = c->N / 2; c->seed = seed;
    c->betas.assign(betas, betas + R);
    c->keys = philox_round_keys((uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32));
    c->ws = ws_layout(L, R);
    const int sms = current_sm_count();
    c->sm_count = sms;                             // xy_attach replaces it by the bound device's
    default_tiles(L, R, c->TY, c->TZ, sms);
    if (!tiles_ok(L, c->TY, c->TZ)) {
        fail(XY_ERR_INVALID_ARG, "xy_create: no valid tile for L=%d (TY=%d TZ=%d)", L, c->TY, c->TZ);
        delete c;
        return nullptr;
    }
    // Measured at L=160: the Metropolis pass is 3 % faster as ONE block of 20 + 1 warps per
    // SM (five compute warps on every scheduler) than as two of 10 + 1; the over-relaxation pass is not.
    if (L == 160 && c->TY == 16) {
        c->TY_met = 32; c->TZ_met = L;
        double best = 1e300;                       // march length for ONE resident block per SM, as in default_tiles
        for (int t = L; t >= 2; --t) {
            if (L % t) continue;
            const long blocks = (long)R * (L / c->TY_met) * (L / t);
            const double cost = (double)((blocks + sms - 1) / sms) * (t + 1.0);
            if (cost < best * 0.999) { best = cost; c->TZ_met = t; }
        }
    }
    // L = 96 and L = 80 (paper sizes): 16 rows x 12 (10) float4 = 6 (5) whole warps -> the compile-time variants
    // (L = 96 with warps of uniform x parity; L = 80: 0.1587 -> 0.1526 ms per step at R = 34 against 20 rows, run-time geometry)
    if ((L == 96 || L == 80) && tiles_ok(L, 16, c->TZ)) {
        c->TY = 16;
        default_tiles_z(L, R, 16, c->TZ, sms);
        // measured at the paper's R = 34 (bench.py --family): L = 80: TZ 16 0.1468 ms per step against 0.1526 (20), 0.1786 (40);
        // L = 96: TZ 24 0.2405 against 0.2594 (32) -- three blocks of these small tiles fit an SM, which the model does not know
        if (R >= 24 && R <= 48) c->TZ = L == 80 ? 16 : 24;
    }
    return c;
}

void xy_destroy(xy_ctx* c) {
    if (!c) return;
    DeviceScope scope;                             // free buffers, stream, events and graph on the device they belong to
    if (c->device >= 0) scope.enter(c->device);
    if (c->own_state && c->d_state) cudaFree(c->d_state);
    if (c->own_ws && c->d_ws) cudaFree(c->d_ws);
    if (c->d_trace) cudaFree(c->d_trace);
    for (auto& s : c->spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
    for (auto e : c->free_events) cudaEventDestroy(e);
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    if (c->own_stream && c->stream) cudaStreamDestroy(c->stream);
    delete c;
}

size_t xy_state_bytes(int L, int R) { return shape_ok(L, R) ? (size_t)R * L * L * L * 4 : 0; }
size_t xy_workspace_bytes(int L, int R) { return shape_ok(L, R) ? ws_layout(L, R).total : 0; }

int xy_attach(xy_ctx* c, void* d_state, void* d_workspace, void* cuda_stream) {
    if (!c) return fail(XY_ERR_INVALID_ARG, "NULL context");
    if (c->attached) return fail(XY_ERR_INVALID_ARG, "xy_attach: context is already attached");
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1) {
        cudaGetLastError();
        return fail(XY_ERR_NO_DEVICE, "xy_attach: no CUDA device; this library has no CPU fallback");
    }
    int dev = 0;
    CK(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(XY_ERR_NO_DEVICE, "xy_attach: device index %d out of range", dev);
    c->device = dev;
    c->sm_count = prop.multiProcessorCount > 0 ? prop.multiProcessorCount : 148;
    if (prop.major < 10) return fail(XY_ERR_NO_DEVICE, "xy_attach: device %s is sm_%d%d; built for sm_100a only", prop.name, prop.major, prop.minor);
    if (((uintptr_t)d_state | (uintptr_t)d_workspace) & 255u) return fail(XY_ERR_INVALID_ARG, "xy_attach: buffers must be 256-byte aligned");
    for (void* p : { d_state, d_workspace }) {        // caller-owned buffers must live on the device this context is bound to
        if (!p) continue;
        cudaPointerAttributes pa;
        if (cudaPointerGetAttributes(&pa, p) != cudaSuccess) { cudaGetLastError(); return fail(XY_ERR_INVALID_ARG, "xy_attach: not a CUDA pointer"); }
        if (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) return fail(XY_ERR_INVALID_ARG, "xy_attach: buffers must be device memory");
        if (pa.type == cudaMemoryTypeDevice && pa.device != dev)
            return fail(XY_ERR_INVALID_ARG, "xy_attach: buffer lives on device %d but the current device is %d", pa.device, dev);
    }
    c->stream = (cudaStream_t)cuda_stream;
    if (c->stream) {                           // a caller's stream must belong to the device this context is bound to
        int sdev = -1;
        if (cudaStreamGetDevice(c->stream, &sdev) != cudaSuccess) {
            cudaGetLastError();
            c->stream = nullptr;
            return fail(XY_ERR_INVALID_ARG, "xy_attach: cuda_stream is not a valid stream");
        }
        if (sdev != dev) {
            c->stream = nullptr;
            return fail(XY_ERR_INVALID_ARG, "xy_attach: the stream belongs to device %d but the current device is %d", sdev, dev);
        }
    }
    if (!c->stream) {                          // the legacy default stream cannot be captured into a graph: use a
        CK(cudaStreamCreate(&c->stream));      // BLOCKING stream of our own, which stays ordered with it
        c->own_stream = true;
    }
    if (d_state) { c->d_state = (float*)d_state; c->own_state = false; }
    else { CK(cudaMalloc(&c->d_state, xy_state_bytes(c->L, c->R))); c->own_state = true; }
    if (d_workspace) { c->d_ws = (char*)d_workspace; c->own_ws = false; }
    else { CK(cudaMalloc(&c->d_ws, c->ws.total)); c->own_ws = true; }
    CK(cudaMemsetAsync(c->d_ws, 0, c->ws.stage, c->stream));     // everything but the staging slot
    c->attached = true;
    c->partials_valid = c->rank_valid = c->slot_valid = false;
    c->launches = 0;
    return upload_labels(c, nullptr);
}

int xy_init_random(xy_ctx* c) {
    ENTER(c);
    const size_t n_quads = (size_t)c->R * c->L * c->L * (c->L / 4);
    {
        LaunchSpan span(c, XY_K_OTHER);
        init_random_kernel<<<grid_for(n_quads, 256), 256, 0, c->stream>>>(c->colour(0), c->colour(1), c->L, c->R, c->keys);
    }
    CK(cudaGetLastError());
    c->partials_valid = c->slot_valid = false;
    return XY_OK;
}

int xy_init_ordered(xy_ctx* c, float theta0) {
    ENTER(c);
    const size_t n = (size_t)c->R * c->N;
    {
        LaunchSpan span(c, XY_K_OTHER);
        fill_kernel<<<grid_for(n, 256), 256, 0, c->stream>>>(c->d_state, n, theta0);
    }
    CK(cudaGetLastError());
    c->partials_valid = c->slot_valid = false;
    return XY_OK;
}

static int convert_state(xy_ctx* c, float* black, float* white, float* natural, int on_device, bool to_split) {
    const int L = c->L;
    const size_t per_slot = (size_t)L * L * (L / 8);
    if (on_device) {
        const size_t n = per_slot * c->R;
        LaunchSpan span(c, XY_K_OTHER);
        if (to_split) convert_kernel<true><<<grid_for(n, 256), 256, 0, c->stream>>>(natural, black, white, L, c->R, 0);
        else convert_kernel<false><<<grid_for(n, 256), 256, 0, c->stream>>>(natural, black, white, L, c->R, 0);
        CK(cudaGetLastError());
        return XY_OK;
    }
    float* stage = c->ws_ptr<float>(c->ws.stage);
    for (int r = 0; r < c->R; ++r) {            // one natural slot at a time through the staging buffer
        float* h = natural + (size_t)r * c->N;
        LaunchSpan span(c, XY_K_OTHER);
        if (to_split) {
            CK(cudaMemcpyAsync(stage, h, c->N * 4, cudaMemcpyHostToDevice, c->stream));
            convert_kernel<true><<<grid_for(per_slot, 256), 256, 0, c->stream>>>(stage, black, white, L, 1, r);
        } else {
            convert_kernel<false><<<grid_for(per_slot, 256), 256, 0, c->stream>>>(stage, black, white, L, 1, r);
            CK(cudaMemcpyAsync(h, stage, c->N * 4, cudaMemcpyDeviceToHost, c->stream));
        }
        CK(cudaGetLastError());
    }
    CK(cudaStreamSynchronize(c->stream));
    return XY_OK;
}

int xy_set_state(xy_ctx* c, const float* natural, int on_device) {
    ENTER(c);
    if (!natural) return fail(XY_ERR_INVALID_ARG, "xy_set_state: NULL pointer");
    c->partials_valid = c->slot_valid = false;
    return convert_state(c, c->colour(0), c->colour(1), const_cast<float*>(natural), on_device, true);
}

int xy_get_state(xy_ctx* c, float* natural, int on_device) {
    ENTER(c);
    if (!natural) return fail(XY_ERR_INVALID_ARG, "xy_get_state: NULL pointer");
    return convert_state(c, c->colour(0), c->colour(1), natural, on_device, false);
}

// Both colour passes of one Metropolis sweep over the slots [slot0, slot0 + n_slots); the caller advances n_met.
static int metropolis_slots(xy_ctx* c, int slot0, int n_slots) {
    if (c->trace && !c->d_trace) CK(cudaMalloc(&c->d_trace, (size_t)c->R * c->N * 4));
    for (int colour = 0; colour < 2; ++colour) {
        SweepParams P = base_params(c, colour);
        P.slot0 = slot0; P.n_slots = n_slots;
        if (c->TY_met && !c->trace && !c->generic && !need_inline_exact(c)) {
            P.TY = c->TY_met; P.TZ = c->TZ_met; P.nTY = c->L / P.TY; P.nTZ = c->L / P.TZ; P.nItems = P.TY * P.W4;
        }
        P.sweep = c->n_met;
        P.trace = c->d_trace;
        const bool inl = need_inline_exact(c);
        int rc = inl ? (c->trace ? launch_sweep<MODE_MET, true, false, true>(c, P) : launch_sweep<MODE_MET, false, false, true>(c, P))
                     : (c->trace ? launch_sweep<MODE_MET, true, false, false>(c, P) : launch_sweep<MODE_MET, false, false, false>(c, P));
        if (rc) return rc;
        if (!inl) {                                  // settle the close decisions before the next pass reads this colour
            FixupParams F;
            memset(&F, 0, sizeof(F));
            F.own = P.own; F.other = P.other; F.L = c->L; F.W = c->L / 2; F.colour = colour; F.R = c->R;
            F.half_n = P.half_n; F.keys = c->keys; F.sweep = c->n_met; F.d_counters = P.d_counters; F.beta32_of_slot = P.beta32_of_slot;
            F.met_acc = P.met_acc; F.exact_count = P.exact_count; F.near_queue = P.near_queue;
            F.near_count = P.near_count; F.near_cap = P.near_cap;
            F.done_ticket = P.near_count + 1; F.overflow_flag = P.near_count + 2;
            {
                LaunchSpan span(c, XY_K_FIXUP);
                CK(launch_chained(chain_pdl(c), met_fixup_kernel, dim3(c->sm_count), dim3(256), 0, c->stream, F));
            }
        }
    }
    return XY_OK;
}

int xy_metropolis_sweep(xy_ctx* c) {
    ENTER(c);
    if (int rc = metropolis_slots(c, 0, c->R)) return rc;
    ++c->n_met;
    c->partials_valid = c->slot_valid = false;
    return XY_OK;
}

// Both colour passes of one over-relaxation sweep over the slots [slot0, slot0 + n_slots); the caller advances n_or.
static int overrelax_slots(xy_ctx* c, bool with_observables, int slot0, int n_slots) {
    for (int colour = 0; colour < 2; ++colour) {
        SweepParams P = base_params(c, colour);
        P.slot0 = slot0; P.n_slots = n_slots;
        const bool fuse = with_observables && colour == 1;      // the white pass sees the final black sites
        int rc = fuse ? launch_sweep<MODE_OR, false, true>(c, P) : launch_sweep<MODE_OR, false, false>(c, P);
        if (rc) return rc;
    }
    return XY_OK;
}

static int overrelax_sweep_impl(xy_ctx* c, bool with_observables) {
    if (int rc = overrelax_slots(c, with_observables, 0, c->R)) return rc;
    ++c->n_or;
    c->partials_valid = with_observables;
    c->rank_valid = c->slot_valid = false;
    return XY_OK;
}

int xy_overrelax_sweep(xy_ctx* c) {
    ENTER(c);
    return overrelax_sweep_impl(c, c->fused != 0);
}

int xy_measure(xy_ctx* c, double* out) {
    ENTER(c);
    if (int rc = run_measure(c, nullptr)) return rc;
    if (out) {
        CK(cudaMemcpyAsync(out, c->ws_ptr<double>(c->ws.obs_rank), (size_t)c->R * 5 * 8, cudaMemcpyDeviceToHost, c->stream));
        return check_near_overflow(c);
    }
    return XY_OK;
}

// One exchange; d_series_row (device, R*5 doubles or null) also receives the by-rank observables the
// decisions were taken on.  When those are not yet reduced to ranks, the final reduction stage and
// the exchange run as ONE kernel.
static int pt_exchange_impl(xy_ctx* c, double* d_series_row) {
    const bool from_slots = !c->partials_valid && c->slot_valid && !d_series_row && !c->device_counters;
    if (!c->partials_valid && !from_slots) {
        SweepParams P = base_params(c, 1);     // own = white, staged = black
        if (int rc = launch_sweep<MODE_MEASURE, false, false>(c, P)) return rc;
        c->partials_valid = true;
        c->rank_valid = false;
    }
    if (!from_slots && (!c->rank_valid || d_series_row || c->device_counters)) {
        const int n_tiles = (c->L / c->TY) * (c->L / c->TZ);
        LaunchSpan span(c, XY_K_PT);
        CK(launch_chained(chain_pdl(c), finalize_pt_kernel, dim3(1), dim3(1024), 0, c->stream,
            (const double*)c->ws_ptr<double>(c->ws.partials), n_tiles, c->R, c->n_pt, c->keys, (const double*)c->ws_ptr<double>(c->ws.betas),
            c->ws_ptr<int>(c->ws.slot_at_rank), c->ws_ptr<double>(c->ws.obs_rank), c->ws_ptr<double>(c->ws.obs_slot),
            d_series_row, c->ws_ptr<double>(c->ws.beta_of_slot), c->ws_ptr<float>(c->ws.beta32),
            c->ws_ptr<unsigned long long>(c->ws.pt_acc),
            c->device_counters ? c->ws_ptr<DeviceCounters>(c->ws.dctr) : (DeviceCounters*)nullptr, c->or_per_mcs));
    } else {
        const int pairs = c->R / 2 + 1;
        LaunchSpan span(c, XY_K_PT);
        pt_exchange_kernel<<<(pairs + 127) / 128, 128, 0, c->stream>>>(
            c->R, c->n_pt, c->keys, c->ws_ptr<double>(c->ws.betas), c->ws_ptr<double>(c->ws.obs_slot),
            c->ws_ptr<int>(c->ws.slot_at_rank), c->ws_ptr<double>(c->ws.beta_of_slot), c->ws_ptr<float>(c->ws.beta32),
            c->ws_ptr<unsigned long long>(c->ws.pt_acc));
    }
    CK(cudaGetLastError());
    ++c->n_pt;
    c->rank_valid = false;                     // the by-rank rows now belong to the previous labelling
    return XY_OK;
}

int xy_measure_stiffness(xy_ctx* c, double* out) {
    ENTER(c);
    if (!out) return fail(XY_ERR_INVALID_ARG, "xy_measure_stiffness: NULL pointer");
    SweepParams P = base_params(c, 1);         // own = white, staged = black
    P.partials = c->ws_ptr<double>(c->ws.partials6);
    if (int rc = launch_sweep<MODE_STIFF, false, false>(c, P)) return rc;
    const int n_tiles = (c->L / c->TY) * (c->L / c->TZ);
    {
        LaunchSpan span(c, XY_K_FINALIZE);
        stiffness_finalize_kernel<<<(c->R + 3) / 4, 128, 0, c->stream>>>(c->ws_ptr<double>(c->ws.partials6), n_tiles, c->R,
                                                                       c->ws_ptr<int>(c->ws.slot_at_rank),
                                                                       c->ws_ptr<double>(c->ws.obs6));
    }
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(out, c->ws_ptr<double>(c->ws.obs6), (size_t)c->R * 6 * 8, cudaMemcpyDeviceToHost, c->stream));
    return check_near_overflow(c);
}

int xy_pt_exchange(xy_ctx* c) {
    ENTER(c);
    return pt_exchange_impl(c, nullptr);
}

// One Monte Carlo step enqueued on the stream [P:30].
static int enqueue_mcs(xy_ctx* c, double* d_series_row) {
    // XY_OPT_SLOT_CHUNK: all colour passes of K slots back to back, chunk after chunk, so that a chunk's spins are still in
    // L2 when its next pass reads them.  The passes of different slots are independent (only the
    // exchange couples replicas), every kernel reads the same step counters: bitwise the same results.
    if (c->slot_chunk > 0 && c->slot_chunk < c->R && !c->trace) {
        for (int s0 = 0; s0 < c->R; s0 += c->slot_chunk) {
            const int n = std::min(c->slot_chunk, c->R - s0);
            if (int rc = metropolis_slots(c, s0, n)) return rc;
            for (int j = 0; j < c->or_per_mcs; ++j)
                if (int rc = overrelax_slots(c, c->fused != 0 && j + 1 == c->or_per_mcs, s0, n)) return rc;
        }
        ++c->n_met; c->n_or += (uint32_t)c->or_per_mcs;
        c->partials_valid = c->fused != 0 && c->or_per_mcs >= 1;
        c->rank_valid = c->slot_valid = false;
        return pt_exchange_impl(c, d_series_row);
    }
    if (int rc = xy_metropolis_sweep(c)) return rc;
    for (int j = 0; j < c->or_per_mcs; ++j)          // only the last sweep's white pass carries the observables
        if (int rc = overrelax_sweep_impl(c, c->fused != 0 && j + 1 == c->or_per_mcs)) return rc;
    return pt_exchange_impl(c, d_series_row);
}

// Captures one step in device-counter mode (the kernels read n_met / n_pt / the series row from the
// workspace and finalize_pt_kernel advances them), so that the same graph can be replayed.
static int build_step_graph(xy_ctx* c, uint64_t key) {
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    const uint32_t n0[3] = { c->n_met, c->n_or, c->n_pt };
    const uint64_t launches0 = c->launches;
    cudaGraph_t graph = nullptr;
    CK(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
    c->device_counters = true;
    const int rc = enqueue_mcs(c, nullptr);
    c->device_counters = false;
    const cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    c->n_met = n0[0]; c->n_or = n0[1]; c->n_pt = n0[2];      // nothing ran: the capture only recorded
    c->graph_launches = c->launches - launches0;             // kernel nodes per step
    c->launches = launches0;
    if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) return fail(XY_ERR_CUDA, "cudaStreamEndCapture failed: %s", cudaGetErrorString(e));
    const cudaError_t e2 = cudaGraphInstantiate(&c->graph_exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e2 != cudaSuccess) { c->graph_exec = nullptr; return fail(XY_ERR_CUDA, "cudaGraphInstantiate failed: %s", cudaGetErrorString(e2)); }
    c->graph_key = key;
    return XY_OK;
}

int xy_mcs(xy_ctx* c, int n_mcs, double* d_series) {
    ENTER(c);
    if (n_mcs < 0) return fail(XY_ERR_INVALID_ARG, "xy_mcs: n_mcs < 0");
    // XY_OPT_RESIDENT: small lattices run all n steps in ONE persistent launch with the spins resident in shared memory
    if (c->resident && !c->trace && n_mcs >= 1) {
        const ResidentPlan& pl = resident_plan(c);
        if (pl.ok) {
            // the kernel counts accepted proposals per thread in 32 bits over one launch: at most 2^24 steps per launch
            // (a thread owns well under 2^7 sites), so xy_get_accept_counts stays exact for any n_mcs
            constexpr int kMaxStepsPerLaunch = 1 << 24;
            for (int done = 0; done < n_mcs; done += kMaxStepsPerLaunch) {
                const int n = std::min(kMaxStepsPerLaunch, n_mcs - done);
                if (const int rc = resident_mcs(c, pl, n, d_series ? d_series + (size_t)done * c->R * 5 : nullptr)) return rc;
            }
            return XY_OK;
        }
    }
    int t = 0;
    // XY_OPT_CUDA_GRAPH: from the second step on, replay one captured graph per step (7 kernel nodes):
    // same kernels, same arithmetic, less launch latency.  The first step runs eagerly (it also sets the
    // kernels' attributes).  Profiling brackets launches with events and the test trace allocates: eager.
    if (c->use_graph && !c->profile && !c->trace && n_mcs >= 3) {
        if (int rc = enqueue_mcs(c, d_series)) return rc;
        t = 1;
        const uint64_t key = 1u | ((uint64_t)c->TY << 1) ^ ((uint64_t)c->TZ << 12) ^ ((uint64_t)c->fused << 23) ^ ((uint64_t)c->generic << 24) ^
                             ((uint64_t)c->or_per_mcs << 25) ^ ((uint64_t)c->slot_chunk << 50) ^ ((uint64_t)c->TY_met << 44) ^ ((uint64_t)need_inline_exact(c) << 36) ^ ((uint64_t)(uintptr_t)c->stream << 37);
        if (!c->graph_exec || c->graph_key != key)
            if (int rc = build_step_graph(c, key)) return rc;
        DeviceCounters v;
        v.n_met = c->n_met; v.n_or = c->n_or; v.n_pt = c->n_pt; v.row = 1u; v.series_base = d_series;
        set_device_counters_kernel<<<1, 1, 0, c->stream>>>(c->ws_ptr<DeviceCounters>(c->ws.dctr), v);
        CK(cudaGetLastError());
        ++c->launches;                             // the counter upload
        for (; t < n_mcs; ++t) {
            // the host counters follow every replay that was enqueued, so that a failing launch leaves them equal
            // to the device's (DeviceCounters) instead of n_mcs - t steps behind
            CK(cudaGraphLaunch(c->graph_exec, c->stream));
            c->n_met += 1u; c->n_or += (uint32_t)c->or_per_mcs; c->n_pt += 1u;
            c->launches += c->graph_launches;
            c->partials_valid = true;              // the step's exchange reduced the final state (labels move, spins do not)
            c->rank_valid = false;
        }
        return XY_OK;
    }
    for (; t < n_mcs; ++t)
        if (int rc = enqueue_mcs(c, d_series ? d_series + (size_t)t * c->R * 5 : nullptr)) return rc;
    return XY_OK;
}

int xy_get_perm(xy_ctx* c, int* p) {
    ENTER(c);
    if (!p) return fail(XY_ERR_INVALID_ARG, "xy_get_perm: NULL pointer");
    CK(cudaMemcpyAsync(p, c->ws_ptr<int>(c->ws.slot_at_rank), c->R * 4, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return XY_OK;
}

int xy_set_perm(xy_ctx* c, const int* p) {
    ENTER(c);
    if (!p) return fail(XY_ERR_INVALID_ARG, "xy_set_perm: NULL pointer");
    std::vector<char> seen(c->R, 0);
    for (int k = 0; k < c->R; ++k) {
        if (p[k] < 0 || p[k] >= c->R || seen[p[k]]) return fail(XY_ERR_INVALID_ARG, "xy_set_perm: not a permutation of 0..R-1");
        seen[p[k]] = 1;
    }
    return upload_labels(c, p);
}

int xy_set_betas(xy_ctx* c, const double* betas) {
    ENTER(c);
    if (!betas) return fail(XY_ERR_INVALID_ARG, "xy_set_betas: NULL pointer");
    for (int k = 0; k < c->R; ++k)
        if (!std::isfinite(betas[k])) return fail(XY_ERR_INVALID_ARG, "xy_set_betas: betas[%d] is not finite", k);
    std::vector<int> perm(c->R);
    CK(cudaMemcpyAsync(perm.data(), c->ws_ptr<int>(c->ws.slot_at_rank), c->R * 4, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    c->betas.assign(betas, betas + c->R);
    return upload_labels(c, perm.data());          // rank k keeps its slot and gets the new beta_k
}

int xy_get_beta_of_slot(xy_ctx* c, double* b) {
    ENTER(c);
    if (!b) return fail(XY_ERR_INVALID_ARG, "xy_get_beta_of_slot: NULL pointer");
    CK(cudaMemcpyAsync(b, c->ws_ptr<double>(c->ws.beta_of_slot), c->R * 8, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return XY_OK;
}

int xy_get_counters(xy_ctx* c, uint32_t n[3]) {
    if (!c || !n) return fail(XY_ERR_INVALID_ARG, "xy_get_counters: NULL argument");
    n[0] = c->n_met; n[1] = c->n_or; n[2] = c->n_pt;
    return XY_OK;
}

int xy_set_counters(xy_ctx* c, const uint32_t n[3]) {
    if (!c || !n) return fail(XY_ERR_INVALID_ARG, "xy_set_counters: NULL argument");
    c->n_met = n[0]; c->n_or = n[1]; c->n_pt = n[2];
    return XY_OK;
}

int xy_get_accept_counts(xy_ctx* c, uint64_t* met, uint64_t* pt) {
    ENTER(c);
    if (met) CK(cudaMemcpyAsync(met, c->ws_ptr<char>(c->ws.met_acc), c->R * 8, cudaMemcpyDeviceToHost, c->stream));
    if (pt && c->R > 1) CK(cudaMemcpyAsync(pt, c->ws_ptr<char>(c->ws.pt_acc), (c->R - 1) * 8, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return XY_OK;
}

int xy_get_exact_path_count(xy_ctx* c, uint64_t* n) {
    ENTER(c);
    if (!n) return fail(XY_ERR_INVALID_ARG, "xy_get_exact_path_count: NULL pointer");
    CK(cudaMemcpyAsync(n, c->ws_ptr<char>(c->ws.exact), 8, cudaMemcpyDeviceToHost, c->stream));
    return check_near_overflow(c);
}

int xy_set_option(xy_ctx* c, int option, int value) {
    if (!c) return fail(XY_ERR_INVALID_ARG, "NULL context");
    switch (option) {
        case XY_OPT_TILE_Y:
            if (!tiles_ok(c->L, value, c->TZ)) return fail(XY_ERR_INVALID_ARG, "XY_OPT_TILE_Y=%d invalid for L=%d", value, c->L);
            c->TY = value; c->TY_met = c->TZ_met = 0; c->partials_valid = c->slot_valid = false; return XY_OK;
        case XY_OPT_TILE_Z:
            if (!tiles_ok(c->L, c->TY, value)) return fail(XY_ERR_INVALID_ARG, "XY_OPT_TILE_Z=%d invalid for L=%d", value, c->L);
            c->TZ = value; c->TY_met = c->TZ_met = 0; c->partials_valid = c->slot_valid = false; return XY_OK;
        case XY_OPT_TRACE: c->trace = value ? 1 : 0; return XY_OK;
        case XY_OPT_FUSED_MEASURE: c->fused = value ? 1 : 0; return XY_OK;
        case XY_OPT_PROFILE: c->profile = value ? 1 : 0; return XY_OK;
        case XY_OPT_GENERIC_KERNEL: c->generic = value ? 1 : 0; return XY_OK;
        case XY_OPT_CUDA_GRAPH: c->use_graph = value ? 1 : 0; return XY_OK;
        case XY_OPT_RESIDENT: c->resident = value ? 1 : 0; return XY_OK;
        case XY_OPT_SLOT_CHUNK:
            if (value < 0) return fail(XY_ERR_INVALID_ARG, "XY_OPT_SLOT_CHUNK=%d out of range", value);
            c->slot_chunk = value; return XY_OK;
        case XY_OPT_OR_PER_MCS:
            if (value < 0 || value > 1000) return fail(XY_ERR_INVALID_ARG, "XY_OPT_OR_PER_MCS=%d out of range", value);
            c->or_per_mcs = value; return XY_OK;
        default: return fail(XY_ERR_INVALID_ARG, "unknown option %d", option);
    }
}

int xy_get_option(xy_ctx* c, int option, int* value) {
    if (!c || !value) return fail(XY_ERR_INVALID_ARG, "NULL argument");
    switch (option) {
        case XY_OPT_TILE_Y: *value = c->TY; return XY_OK;
        case XY_OPT_TILE_Z: *value = c->TZ; return XY_OK;
        case XY_OPT_TRACE: *value = c->trace; return XY_OK;
        case XY_OPT_FUSED_MEASURE: *value = c->fused; return XY_OK;
        case XY_OPT_PROFILE: *value = c->profile; return XY_OK;
        case XY_OPT_GENERIC_KERNEL: *value = c->generic; return XY_OK;
        case XY_OPT_OR_PER_MCS: *value = c->or_per_mcs; return XY_OK;
        case XY_OPT_CUDA_GRAPH: *value = c->use_graph; return XY_OK;
        case XY_OPT_RESIDENT: *value = c->resident; return XY_OK;
        case XY_OPT_SLOT_CHUNK: *value = c->slot_chunk; return XY_OK;
        default: return fail(XY_ERR_INVALID_ARG, "unknown option %d", option);
    }
}

int xy_get_kernel_times(xy_ctx* c, double* ms, uint64_t* n) {
    ENTER(c);
    if (!ms || !n) return fail(XY_ERR_INVALID_ARG, "xy_get_kernel_times: NULL pointer");
    CK(cudaStreamSynchronize(c->stream));
    for (auto& s : c->spans) {
        float t = 0.f;
        CK(cudaEventElapsedTime(&t, s.a, s.b));
        c->k_ms[s.cls] += (double)t;
        c->k_n[s.cls] += 1;
        c->free_events.push_back(s.a);
        c->free_events.push_back(s.b);
    }
    c->spans.clear();
    for (int k = 0; k < XY_NUM_KERNEL_CLASSES; ++k) { ms[k] = c->k_ms[k]; n[k] = c->k_n[k]; c->k_ms[k] = 0.0; c->k_n[k] = 0; }
    return XY_OK;
}

int xy_get_resident_plan(xy_ctx* c, int out[6]) {
    ENTER(c);
    if (!out) return fail(XY_ERR_INVALID_ARG, "xy_get_resident_plan: NULL pointer");
    const ResidentPlan& pl = resident_plan(c);
    // XY_OPT_TRACE forces the per-pass kernels
    out[0] = pl.ok && c->resident && !c->trace ? 1 : 0; out[1] = pl.G; out[2] = pl.C; out[3] = pl.threads; out[4] = pl.grid; out[5] = (int)pl.smem;
    return XY_OK;
}

int xy_get_launch_count(xy_ctx* c, uint64_t* n) {
    if (!c || !n) return fail(XY_ERR_INVALID_ARG, "NULL argument");
    *n = c->launches;
    return XY_OK;
}

int xy_synchronize(xy_ctx* c) {
    ENTER(c);
    return check_near_overflow(c);
}

int xy_debug_get_trace(xy_ctx* c, float* natural) {
    ENTER(c);
    if (!natural) return fail(XY_ERR_INVALID_ARG, "xy_debug_get_trace: NULL pointer");
    if (!c->d_trace) return fail(XY_ERR_INVALID_ARG, "xy_debug_get_trace: no trace recorded (set XY_OPT_TRACE before the sweep)");
    return convert_state(c, c->d_trace, c->d_trace + (size_t)c->R * c->half_n, natural, 0, false);
}

int xy_debug_sincos(const float* d_x, float* d_cos, float* d_sin, size_t n, void* stream) {
    if (!d_x || !d_cos || !d_sin) return fail(XY_ERR_INVALID_ARG, "xy_debug_sincos: NULL pointer");
    debug_sincos_kernel<<<grid_for(n, 256), 256, 0, (cudaStream_t)stream>>>(d_x, d_cos, d_sin, n);
    CK(cudaGetLastError());
    return XY_OK;
}

int xy_debug_sincos64(const double* d_x, double* d_cos, double* d_sin, size_t n, void* stream) {
    if (!d_x || !d_cos || !d_sin) return fail(XY_ERR_INVALID_ARG, "xy_debug_sincos64: NULL pointer");
    debug_sincos64_kernel<<<grid_for(n, 256), 256, 0, (cudaStream_t)stream>>>(d_x, d_cos, d_sin, n);
    CK(cudaGetLastError());
    return XY_OK;
}

int xy_debug_atan2(const float* d_y, const float* d_x, float* d_phi, size_t n, void* stream) {
    if (!d_x || !d_y || !d_phi) return fail(XY_ERR_INVALID_ARG, "xy_debug_atan2: NULL pointer");
    debug_atan2_kernel<<<grid_for(n, 256), 256, 0, (cudaStream_t)stream>>>(d_y, d_x, d_phi, n);
    CK(cudaGetLastError());
    return XY_OK;
}

int xy_debug_philox(const uint32_t* d_ctr, uint32_t key0, uint32_t key1, uint32_t* d_out, size_t n, void* stream) {
    if (!d_ctr || !d_out) return fail(XY_ERR_INVALID_ARG, "xy_debug_philox: NULL pointer");
    debug_philox_kernel<<<grid_for(n, 256), 256, 0, (cudaStream_t)stream>>>(d_ctr, philox_round_keys(key0, key1), d_out, n);
    CK(cudaGetLastError());
    return XY_OK;
}

}  // extern "C"

// ---- xy_measure_static: the observable reduction with its scratch compiled into the library ------------------
// For callers that may not allocate (include/xy.h says who and why).  The per-tile partial sums that travel from
// the first kernel (sweep_kernel in MODE_MEASURE) to the second live in this file-scope array instead of a
// workspace: 1 MiB that every device holds from the load of this module until the process exits.
// NOTE for maintainers: in HOST code the name `xy_static_scratch` is only a handle for the runtime, not a device
// address -- never pass it to a kernel.  static_setup() below asks the runtime for the real address once per
// device (cudaGetSymbolAddress, with that device current) and the launch code passes THAT pointer.  Device code
// (measure_finalize_static_kernel) may and does name the array directly.
static __device__ __align__(256) unsigned char xy_static_scratch[XY_STATIC_SCRATCH_BYTES];

namespace {

// Second stage of the static variant: one warp per SLOT sums that slot's tile partials out of the built-in array
// in the same fixed order as finalize_rank (lane l takes tiles l, l+32, ..., then a shuffle tree); lane 0 writes
// the five observables.  No permutation: the caller has no context, rows are by slot.
__global__ void measure_finalize_static_kernel(int n_tiles, int R, double* __restrict__ out_slot) {
    const int slot = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (slot >= R) return;
    const double* __restrict__ partials = reinterpret_cast<const double*>(xy_static_scratch);
    double v[3] = { 0.0, 0.0, 0.0 };
    for (int t = lane; t < n_tiles; t += 32)
        for (int c = 0; c < 3; ++c) v[c] += partials[((size_t)slot * n_tiles + t) * 3 + c];
    for (int c = 0; c < 3; ++c)
        for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
    if (lane == 0) {
        const double m2 = v[1] * v[1] + v[2] * v[2];
        out_slot[5 * slot + 0] = v[0]; out_slot[5 * slot + 1] = v[1]; out_slot[5 * slot + 2] = v[2];
        out_slot[5 * slot + 3] = m2;   out_slot[5 * slot + 4] = m2 * m2;
    }
}

// Per-device set-up of the static variant, done by the first xy_measure_static call that finds the device current:
// the device address of the array on THIS device and the first kernel's dynamic-shared-memory opt-in.  Neither
// allocates; neither is stream work (hence "first call before any stream capture" in xy.h).
struct StaticDevice { bool ready = false; double* scratch = nullptr; };
StaticDevice g_static_dev[kMaxDevices];
std::mutex g_static_mutex;

int static_setup(int dev, double** scratch) {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice& s = g_static_dev[dev];
    if (!s.ready) {
        int major = 0;
        CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        if (major < 10) return fail(XY_ERR_NO_DEVICE, "xy_measure_static: device %d is sm_%dx; built for sm_100a only", dev, major);
        void* p = nullptr;
        CK(cudaGetSymbolAddress(&p, xy_static_scratch));       // valid for the device that is current now, i.e. `dev`
        if (!p) return fail(XY_ERR_CUDA, "xy_measure_static: cudaGetSymbolAddress returned a null address");
        CK(cudaFuncSetAttribute(sweep_kernel<MODE_MEASURE, false, false, false, 0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        s.scratch = static_cast<double*>(p);
        s.ready = true;
    }
    *scratch = s.scratch;
    return XY_OK;
}

}  // namespace

extern "C" int xy_measure_static(const float* d_state, int L, int R, double* d_out, void* cuda_stream) {
    if (!shape_ok(L, R)) return fail(XY_ERR_INVALID_ARG, "xy_measure_static: need L %% 8 == 0, 8 <= L <= 1024, 1 <= R <= 65535 (got L=%d R=%d)", L, R);
    int TY = 0, TZ = 0;
    default_tiles(L, R, TY, TZ);
    if (!tiles_ok(L, TY, TZ)) return fail(XY_ERR_INVALID_ARG, "xy_measure_static: no valid tile for L=%d (TY=%d TZ=%d)", L, TY, TZ);
    // the whole size check comes before anything touches the device: a shape beyond the built-in array is refused
    const size_t n_tiles = (size_t)(L / TY) * (size_t)(L / TZ);
    const size_t need = (size_t)R * n_tiles * 3 * sizeof(double);
    if (need > (size_t)XY_STATIC_SCRATCH_BYTES)
        return fail(XY_ERR_INVALID_ARG,
                    "xy_measure_static: L=%d R=%d needs %zu bytes of scratch (24 x %d replicas x %zu tiles) but the built-in array holds %zu; "
                    "use xy_measure on a context for this size", L, R, need, R, n_tiles, (size_t)XY_STATIC_SCRATCH_BYTES);
    if (!d_state || !d_out) return fail(XY_ERR_INVALID_ARG, "xy_measure_static: NULL pointer");
    if (((uintptr_t)d_state & 15u) || ((uintptr_t)d_out & 7u)) return fail(XY_ERR_INVALID_ARG, "xy_measure_static: d_state must be 16-byte and d_out 8-byte aligned");
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1) {
        cudaGetLastError();
        return fail(XY_ERR_NO_DEVICE, "xy_measure_static: no CUDA device; this library has no CPU fallback");
    }
    int dev = 0;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(XY_ERR_NO_DEVICE, "xy_measure_static: device index %d out of range", dev);
    for (const void* p : { (const void*)d_state, (const void*)d_out }) {      // both must be device memory of the current device
        cudaPointerAttributes pa;
        if (cudaPointerGetAttributes(&pa, p) != cudaSuccess) { cudaGetLastError(); return fail(XY_ERR_INVALID_ARG, "xy_measure_static: not a CUDA pointer"); }
        if (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) return fail(XY_ERR_INVALID_ARG, "xy_measure_static: d_state and d_out must be device memory");
        if (pa.type == cudaMemoryTypeDevice && pa.device != dev)
            return fail(XY_ERR_INVALID_ARG, "xy_measure_static: a buffer lives on device %d but the current device is %d", pa.device, dev);
    }
    double* scratch = nullptr;
    if (const int rc = static_setup(dev, &scratch)) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;

    const size_t half_n = (size_t)L * L * L / 2;
    SweepParams P;
    memset(&P, 0, sizeof(P));
    P.own = const_cast<float*>(d_state) + (size_t)R * half_n;      // own = white (MODE_MEASURE stores nothing to it), staged = black
    P.other = d_state;
    P.L = L; P.W = L / 2; P.W4 = L / 8;
    P.TY = TY; P.TZ = TZ; P.nTY = L / TY; P.nTZ = L / TZ;
    P.colour = 1;
    P.slot0 = 0; P.n_slots = R;
    P.nItems = TY * P.W4;
    P.half_n = (unsigned int)half_n;
    P.partials = scratch;                                          // the device address from cudaGetSymbolAddress, never the symbol
    const int threads = (P.nItems + 31) / 32 * 32 + 32;            // compute warps + the auxiliary warp
    sweep_kernel<MODE_MEASURE, false, false, false, 0, 0><<<dim3(P.nTY * P.nTZ, R), threads, sweep_smem_bytes(L, TY), stream>>>(P);
    CK(cudaGetLastError());
    measure_finalize_static_kernel<<<(R + 3) / 4, 128, 0, stream>>>((int)n_tiles, R, d_out);
    CK(cudaGetLastError());
    return XY_OK;
}
