// sdtw.cu -- host side of libsdtw: argument checks, schedule/workspace plan, kernel launches, the C ABI of
// include/sdtw.h.  The arithmetic is in sdtw_kernels.cuh.  No CPU fallback exists: a device that is not sm_100 is
// rejected with SDTW_ERR_UNSUPPORTED.
#include "sdtw.h"
#include "sdtw_debug.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <mutex>
#include <numeric>
#include <vector>

#include "sdtw_kernels.cuh"
#include "sdtw_reverse.cuh"
#include "dtw_kernel.cuh"

namespace {
using namespace sdtw;

thread_local int g_last_cuda_error = 0;
std::mutex g_mutex;
uint64_t g_launches = 0;
struct UserWs { void* ptr = nullptr; size_t bytes = 0; };
UserWs g_user_ws[64];         // caller-registered workspace, one per device (sdtw_set_workspace)
size_t g_ws_limit = 0;        // sdtw_set_workspace_limit: 0 = what the device has free
// instrumentation / tuning switches of include/sdtw_debug.h: per calling thread, so that one thread's measurement
// settings never change another thread's launch
thread_local bool g_profile = false;
thread_local int g_dense_reverse = 0;
thread_local int g_forward_rings = 1;       // 0: never, 1: when the boundary columns would be large, 2: whenever possible (sdtw_set_forward_rings)
thread_local int g_reverse_kernel = -1;    // -1 = automatic, 0 = backward_kernel, 1 = reverse_kernel (sdtw_set_reverse_kernel)
thread_local int g_unit_strips = 0;        // 0 = automatic (sdtw_set_schedule)
thread_local int g_tail_strips = -1, g_tail_unit = 0;   // -1 = automatic (sdtw_set_schedule_tail)
thread_local const unsigned long long* g_last_stats = nullptr;   // device address of the last evaluation's reverse statistics
thread_local uint64_t g_last_stats_gen = 0;   // ... valid while no workspace has been freed since (g_ws_gen)
uint64_t g_ws_gen = 1;
thread_local int g_last_waves = 0;          // waves the last sdtw_value_grad[_ex] / sdtw_barycenter[_ex] call of this thread was split into
size_t g_plan_cap = 32;                     // plans kept (LRU); raised to hold every sub-plan of a call split into many waves

// CUDA events bracketing the phases of one evaluation: start | prologue | forward | reverse | small kernels.
// Owned by a ProfScope until the evaluation has been enqueued completely; an early return destroys them.
struct ProfRec { cudaEvent_t e[5] = {nullptr, nullptr, nullptr, nullptr, nullptr}; };
thread_local std::vector<ProfRec> g_prof;
struct ProfScope {
    ProfRec rec;
    bool on = false, kept = false;
    int begin(bool enable) {
        on = enable;
        if (!on) return cudaSuccess;
        for (auto& e : rec.e) { cudaError_t r = cudaEventCreate(&e); if (r != cudaSuccess) return (int)r; }
        return cudaSuccess;
    }
    int mark(int i, cudaStream_t s) { return on ? (int)cudaEventRecord(rec.e[i], s) : (int)cudaSuccess; }
    void keep() { if (on) { g_prof.push_back(rec); kept = true; } }
    ~ProfScope() { if (on && !kept) for (auto& e : rec.e) if (e) cudaEventDestroy(e); }
};

#define CUDA_TRY(expr)                                   \
    do {                                                 \
        cudaError_t _e = (expr);                         \
        if (_e != cudaSuccess) {                         \
            g_last_cuda_error = (int)_e;                 \
            return SDTW_ERR_CUDA;                        \
        }                                                \
    } while (0)

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ---- workspace layout -------------------------------------------------------------------------------------------
struct Layout {
    int NS = 0;                 // strips per pair
    long long items = 0;
    size_t off_stats = 0;
    int ring_units = 0;         // forward-only ring mode: strips per unit (0: one full boundary column per strip)
    int ring_ctas = 0;          // CTAs the ring buffers are sized for
    size_t off_ring = 0, off_ring_prog = 0;
    size_t off_counters = 0, off_prog_b = 0, off_hint_b = 0, off_ready_b = 0, off_VP = 0, off_Xs = 0, off_Zs = 0, off_VS = 0, off_ES = 0, off_CK = 0,
           off_Gk = 0, off_G = 0, off_Zt = 0, off_Vt = 0, off_scal = 0;   // last four: line-search scratch
    size_t sync_bytes = 0;      // counters + stats + prog_b: cleared before every evaluation
    size_t vs_bytes = 0;        // VS: preset to the sentinel pattern before every evaluation
    size_t total = 0;
    std::vector<PairMeta> pm;   // schedule order
};

template <int D> constexpr int fwd_warps() { return D <= 2 ? 32 : 16; }   // warps per CTA of the forward kernel = strips per unit
inline int fwd_warps_rt(int d) { return d <= 2 ? 32 : 16; }

// ring_sms > 0: forward-only Soft-DTW call without a band on a device with that many SMs.  If the problem has more
// strips than resident forward warps (the throughput regime), strip-boundary values travel through per-warp rings inside
// a unit and only the unit boundaries keep a full column (sdtw_kernels.cuh, forward_kernel): O(chunks) live state per
// resident strip instead of a column per strip ("skipped entirely when out_grad == NULL").
int build_layout(int64_t m, int32_t d, const int64_t* offsets, int32_t N, bool want_grad, Layout& L, int vs_words = 1,
                 int ring_sms = 0) {
    const int max_d = (vs_words == 2) ? SDTW_DTW_MAX_D : SDTW_MAX_D;   // vs_words == 2: the DTW / Sub-DTW kernels
    if (!offsets || m < 1 || d < 1 || N < 1) return SDTW_ERR_INVALID_ARG;
    if (offsets[0] != 0) return SDTW_ERR_INVALID_ARG;
    for (int k = 0; k < N; ++k)
        if (offsets[k + 1] <= offsets[k]) return SDTW_ERR_INVALID_ARG;
    if (d > max_d || m >= (1LL << 30) || N >= (1 << 24)) return SDTW_ERR_UNSUPPORTED;
    for (int k = 0; k < N; ++k)
        if (offsets[k + 1] - offsets[k] >= (1LL << 30)) return SDTW_ERR_UNSUPPORTED;
    const int strip_cols = (vs_words == 2) ? 32 * ((d <= 2) ? dtw_w<1>() : dtw_w<4>()) : SW;   // DTW kernels: dtw_kernel.cuh
    L.NS = (int)((m + strip_cols - 1) / strip_cols);
    L.items = (long long)N * L.NS;
    if (L.items >= (1LL << 31)) return SDTW_ERR_UNSUPPORTED;
    // schedule order: longest cycle first (stable), so the shortest sweeps fill the tail
    std::vector<int> order(N);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) {
        return (offsets[a + 1] - offsets[a]) > (offsets[b + 1] - offsets[b]);
    });
    // (the DTW kernels, vs_words == 2, have a CTA-full of 32 warps only at d <= 2: more channels keep a column per strip)
    // ring_sms < 0: rings whenever the problem has more strips than resident warps.  ring_sms > 0: only when, besides,
    // a column per strip would take more than RING_MIN_COLUMN_BYTES: the ring layout hands out uniform units (a small
    // unit costs a column), and without the small units at the end of the queue a launch of a few hundred pairs drains
    // badly (100 pairs of 30k, forward only: 62.5 ms with columns, 70.3 ms with rings; 1000 pairs: 577 / 584 ms).
    constexpr long long RING_MIN_COLUMN_BYTES = 6LL << 30;
    const int rsms = ring_sms < 0 ? -ring_sms : ring_sms;
    if (rsms > 0 && !want_grad && (vs_words == 1 ? d <= SDTW_MAX_D : d <= 2) &&
        (long long)L.NS * N > (long long)rsms * fwd_warps_rt(d)) {
        long long column_bytes = 0;
        for (int k = 0; k < N; ++k) {
            const long long n = offsets[k + 1] - offsets[k];
            const long long C = ((n + RP - 1) / RP + 31 + CH - 1) / CH;
            column_bytes += 4LL * vs_words * (VS_PAD + C * CROWS) * L.NS;
        }
        if (ring_sms < 0 || column_bytes > RING_MIN_COLUMN_BYTES) {
            L.ring_units = fwd_warps_rt(d);
            L.ring_ctas = rsms;
        }
    }
    const int cols_per_pair = L.ring_units ? (L.NS + L.ring_units - 1) / L.ring_units - 1 : L.NS;   // boundary columns kept
    L.pm.resize(N);
    long long vs_floats = 0, ck_floats = 0;
    for (int ps = 0; ps < N; ++ps) {
        const int k = order[ps];
        PairMeta& pm = L.pm[ps];
        pm.k = k;
        pm.x_off = offsets[k];
        pm.n = (int)(offsets[k + 1] - offsets[k]);
        pm.C = ((pm.n + RP - 1) / RP + 31 + CH - 1) / CH;
        pm.vs_stride = vs_words * (VS_PAD + pm.C * CROWS);   // 32-bit words per strip (the DTW kernel keeps 2 per row)
        pm.vs_off = vs_floats;
        vs_floats += (long long)pm.vs_stride * cols_per_pair;
        pm.ck_stride = (long long)(pm.C * (CH / TR) + 1) * CK_FLOATS;
        pm.ck_off = ck_floats;
        if (want_grad) ck_floats += pm.ck_stride * L.NS;
    }
    size_t o = 0;
    L.off_counters = o; o += 128;
    L.off_stats = o;    o += 128;
    L.off_prog_b = o;   o += align_up((size_t)L.items * 4, 256);
    L.off_hint_b = o;   o += align_up((size_t)L.items * 4, 256);
    L.off_ready_b = o;  o += want_grad ? align_up((size_t)L.items * 4, 256) : 0;
    if (L.ring_units) {         // zeroed with the counters: a ring entry is valid when its tag (>= 1) is the expected one
        L.off_ring = o;      o += (size_t)L.ring_ctas * L.ring_units * (vs_words == 2 ? DTW_RING_ENTRIES * 32 : RING_ENTRIES * 16);
        L.off_ring_prog = o; o += align_up((size_t)L.ring_ctas * L.ring_units * 4, 256);
    }
    L.sync_bytes = o;
    L.off_VP = o;       o += align_up((size_t)L.items * 8, 256);
    L.off_Xs = o;       o += align_up((size_t)offsets[N] * (size_t)d * 4, 256);
    L.off_Zs = o;       o += align_up((size_t)m * (size_t)d * 4, 256);
    L.vs_bytes = align_up((size_t)vs_floats * 4, 256);
    L.off_VS = o;       o += L.vs_bytes;
    if (want_grad) {
        L.off_ES = o;   o += L.vs_bytes;
        L.off_CK = o;   o += align_up((size_t)ck_floats * 4, 256);
        L.off_Gk = o;   o += align_up((size_t)N * (size_t)m * (size_t)d * 4, 256);
        L.off_G = o;    o += align_up((size_t)m * (size_t)d * 4, 256);
        L.off_Zt = o;   o += align_up((size_t)m * (size_t)d * 4, 256);
        L.off_Vt = o;   o += align_up((size_t)N * 4, 256);
        L.off_scal = o; o += 256;
    }
    L.total = o;
    return SDTW_OK;
}

// ---- device / plan cache ----------------------------------------------------------------------------------------
struct DeviceInfo { int dev = -1, sms = 0, cc_major = 0; bool ok = false; };

int get_device(DeviceInfo& di) {
    static DeviceInfo cache[64];
    static std::mutex cache_mutex;                  // the *_workspace_bytes queries come here without g_mutex
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return SDTW_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> cache_lock(cache_mutex);
    if (!cache[dev].ok) {
        cudaDeviceProp prop;
        CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
        cache[dev].dev = dev;
        cache[dev].sms = prop.multiProcessorCount;
        cache[dev].cc_major = prop.major;
        cache[dev].ok = true;
    }
    di = cache[dev];
    if (di.cc_major != 10) return SDTW_ERR_UNSUPPORTED;
    return SDTW_OK;
}

// Instantiated CUDA graph of a whole call on a small problem (launch-bound: a barycenter iteration on configs[0] is
// four kernels of a few microseconds each).  Keyed by everything the captured launches bake in.
struct GraphKey {
    const void *Z, *X, *values, *objective, *grad, *ws;
    int32_t iters, band;
    float gamma, step;
    bool operator==(const GraphKey& o) const { return std::memcmp(this, &o, sizeof(GraphKey)) == 0; }
};
struct GraphEntry { GraphKey key; cudaGraphExec_t exec = nullptr; uint64_t launches = 0, stamp = 0; };

struct Plan {
    int dev = -1;
    std::vector<GraphEntry> graphs;
    std::vector<GraphKey> seen;   // keys met once: a graph is built when a key comes back (a caller that never repeats pays nothing)
    long long cells = 0;          // sum_k n_k * m
    int64_t m = 0;
    int32_t d = 0, N = 0;
    bool want_grad = false;
    int ring_ok = 0;              // forward-only call without a band: 1 = the layout may use rings, 2 = rings whenever possible
    int vs_words = 1;
    std::vector<int64_t> offsets;
    std::vector<float> weights;   // caller order; empty = unweighted
    std::vector<float> weights_sched;   // schedule order (source of the upload; lives as long as the plan)
    Layout L;
    PairMeta* d_pm = nullptr;
    float* d_w = nullptr;         // weights in schedule order (null when unweighted)
    cudaEvent_t uploaded = nullptr;
    uint64_t stamp = 0;
};
std::vector<Plan*> g_plans;
uint64_t g_stamp = 0;

// the cached plan of this problem, or null
Plan* find_plan(int dev, int64_t m, int32_t d, const int64_t* offsets, int32_t N, const float* weights, bool want_grad,
                int vs_words, int ring_ok) {
    for (Plan* pl : g_plans) {
        if (pl->dev == dev && pl->m == m && pl->d == d && pl->N == N && pl->want_grad == want_grad &&
            pl->vs_words == vs_words && pl->ring_ok == ring_ok &&
            std::memcmp(pl->offsets.data(), offsets, sizeof(int64_t) * (size_t)(N + 1)) == 0 &&
            (weights ? (!pl->weights.empty() && std::memcmp(pl->weights.data(), weights, sizeof(float) * (size_t)N) == 0)
                     : pl->weights.empty()))
            return pl;
    }
    return nullptr;
}

int get_plan(const DeviceInfo& di, int64_t m, int32_t d, const int64_t* offsets, int32_t N, const float* weights, bool want_grad,
             cudaStream_t stream, Plan** out, int vs_words = 1, int ring_ok = 0) {
    const int dev = di.dev;
    if (Plan* hit = find_plan(dev, m, d, offsets, N, weights, want_grad, vs_words, ring_ok)) {
        hit->stamp = ++g_stamp;
        CUDA_TRY(cudaStreamWaitEvent(stream, hit->uploaded, 0));
        *out = hit;
        return SDTW_OK;
    }
    Plan* pl = new Plan();
    int rc = build_layout(m, d, offsets, N, want_grad, pl->L, vs_words, ring_ok == 2 ? -di.sms : (ring_ok ? di.sms : 0));
    if (rc != SDTW_OK) { delete pl; return rc; }
    pl->vs_words = vs_words;
    pl->ring_ok = ring_ok;
    pl->dev = dev; pl->m = m; pl->d = d; pl->N = N; pl->want_grad = want_grad;
    pl->offsets.assign(offsets, offsets + N + 1);
    pl->cells = (long long)offsets[N] * m;
    cudaError_t e = cudaMalloc(&pl->d_pm, sizeof(PairMeta) * (size_t)N);
    if (e == cudaSuccess) e = cudaMemcpyAsync(pl->d_pm, pl->L.pm.data(), sizeof(PairMeta) * (size_t)N, cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess && weights) {                 // eq. 7 weights, permuted to schedule order
        pl->weights.assign(weights, weights + N);
        pl->weights_sched.resize((size_t)N);
        for (int ps = 0; ps < N; ++ps) pl->weights_sched[ps] = weights[pl->L.pm[ps].k];
        e = cudaMalloc(&pl->d_w, sizeof(float) * (size_t)N);
        if (e == cudaSuccess) e = cudaMemcpyAsync(pl->d_w, pl->weights_sched.data(), sizeof(float) * (size_t)N, cudaMemcpyHostToDevice, stream);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&pl->uploaded, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventRecord(pl->uploaded, stream);
    if (e != cudaSuccess) {
        g_last_cuda_error = (int)e;
        if (pl->d_pm) cudaFree(pl->d_pm);
        if (pl->d_w) cudaFree(pl->d_w);
        delete pl;
        return SDTW_ERR_CUDA;
    }
    pl->stamp = ++g_stamp;
    if (g_plans.size() >= g_plan_cap) {   // evict the least recently used plan
        auto it = std::min_element(g_plans.begin(), g_plans.end(), [](Plan* a, Plan* b) { return a->stamp < b->stamp; });
        cudaFree((*it)->d_pm);
        if ((*it)->d_w) cudaFree((*it)->d_w);
        for (auto& ge : (*it)->graphs) cudaGraphExecDestroy(ge.exec);
        cudaEventDestroy((*it)->uploaded);
        delete *it;
        g_plans.erase(it);
    }
    g_plans.push_back(pl);
    *out = pl;
    return SDTW_OK;
}

// ---- kernel launch helpers --------------------------------------------------------------------------------------
template <typename K>
int persistent_grid(K kernel, int smem_bytes, int sms, long long items, int* grid) {
    CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
    int occ = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, WARPS * 32, smem_bytes));
    if (occ < 1) return SDTW_ERR_UNSUPPORTED;
    long long want = (items + WARPS - 1) / WARPS;
    long long cap = (long long)sms * occ;
    *grid = (int)std::max(1LL, std::min(want, cap));
    return SDTW_OK;
}

template <int D, bool CKPT>
int launch_forward_t(Params P, int sms, cudaStream_t stream, int ring_ctas) {
    constexpr int FW = fwd_warps<D>();
    const int smem = FW * fwd_smem_floats<D>() * 4;
    auto kernel = forward_kernel<D, CKPT, FW>;
    CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    int occ = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, FW * 32, smem));
    if (occ < 1) return SDTW_ERR_UNSUPPORTED;
    // Strips per unit.  Throughput regime (more strips than resident warps): a unit fills a CTA, so a strip and its
    // producer share an SM.  Latency regime (every strip resident at once: few or short pairs): one strip per unit
    // spreads each pair's dependency chain over as many SMs as possible.
    const bool all_resident = (long long)P.NS * P.N <= (long long)sms * occ * FW;
    P.unit_strips = (g_unit_strips > 0) ? std::min(g_unit_strips, FW) : (all_resident ? 1 : FW);
    if (P.ring) {               // ring layout (forward only): uniform CTA-full units, whatever the tuning hooks say
        P.unit_strips = FW;
        P.tail_unit = FW;
        P.tail_from = P.NS / FW * FW;
    } else {
        const int US = P.unit_strips;
        // The queue ends with small units: the last one-to-two CTA-fulls of strips of every pair go out 4 at a time, so
        // the sweeps still running when the queue empties are spread over all SMs (cfg 4 forward 68.3 -> 66.6 ms).
        const bool small_tail = !all_resident && US > 4 && P.NS >= 2 * US;
        int tail = (g_tail_strips >= 0) ? g_tail_strips : (small_tail ? P.NS % US + US : 0);
        P.tail_unit = (g_tail_unit > 0) ? std::min(g_tail_unit, US) : (small_tail && g_tail_strips < 0 ? 4 : US);
        P.tail_from = std::max(0, (P.NS - tail) / US * US);                 // multiple of US
        if (P.tail_unit == US) P.tail_from = P.NS / US * US;               // uniform: the remainder group only
    }
    const long long units = ((long long)(P.tail_from / P.unit_strips) +
                             (P.NS - P.tail_from + P.tail_unit - 1) / P.tail_unit) * P.N;
    const long long ctas = P.ring ? std::min((long long)sms * occ, (long long)ring_ctas) : (long long)sms * occ;
    const int grid = (int)std::max(1LL, std::min(units, ctas));
    kernel<<<grid, FW * 32, smem, stream>>>(P);
    ++g_launches;
    CUDA_TRY(cudaGetLastError());
    return SDTW_OK;
}

template <int D>
int launch_forward(const Params& P, bool ckpt, int sms, cudaStream_t stream, int ring_ctas) {
    return ckpt ? launch_forward_t<D, true>(P, sms, stream, 0) : launch_forward_t<D, false>(P, sms, stream, ring_ctas);
}

// Two reverse kernels, same arithmetic.  reverse_kernel (sdtw_reverse.cuh: a CTA of 4 warps per strip, the recompute off
// the dependency chain) wins wherever a pair's chain of strips bounds the pass: few pairs, or most chunks skipped.
// backward_kernel (one warp per strip, four times as many strips in flight) wins when the pass is bound by throughput:
// the dense mode, or many more pairs than SMs.  Measured on a B200, reverse pass of one evaluation, new / old kernel:
// N = 25 / 50 / 100 pairs of 30k: 6.7 / 8.0 / 9.4 ms against 12.1 / 12.7 / 13.5 ms; 200 pairs of 15k: 5.5 against 7.1 ms;
// 400 pairs of 15k: 9.0 against 8.6 ms (gamma = 1: 15.8 against 11.7 ms); dense, 100 pairs of 30k: 184 against 138 ms.
constexpr int LATENCY_KERNEL_MAX_PAIRS = 256;

template <int D>
int launch_reverse(const Params& P, int sms, cudaStream_t stream) {
    const int smem = rev_smem_bytes<D>();
    CUDA_TRY(cudaFuncSetAttribute(reverse_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    int occ = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, reverse_kernel<D>, RW * 32, smem));
    if (occ < 1) return SDTW_ERR_UNSUPPORTED;
    const int grid = (int)std::max(1LL, std::min((long long)P.num_items, (long long)sms * occ));
    reverse_kernel<D><<<grid, RW * 32, smem, stream>>>(P);
    ++g_launches;
    CUDA_TRY(cudaGetLastError());
    return SDTW_OK;
}

template <int D>
int launch_backward(const Params& P, int sms, cudaStream_t stream) {
    const bool latency = (g_reverse_kernel >= 0) ? (g_reverse_kernel == 1) : (!P.dense_reverse && P.N <= LATENCY_KERNEL_MAX_PAIRS);
    if (latency) return launch_reverse<D>(P, sms, stream);
    const int smem = WARPS * bwd_smem_floats<D>() * 4;
    int grid = 1;
    int rc = persistent_grid(backward_kernel<D>, smem, sms, P.num_items, &grid);
    if (rc) return rc;
    backward_kernel<D><<<grid, WARPS * 32, smem, stream>>>(P);
    ++g_launches;
    CUDA_TRY(cudaGetLastError());
    return SDTW_OK;
}

int dispatch_forward(int d, const Params& P, bool ckpt, int sms, cudaStream_t s, int ring_ctas) {
    switch (d) {
        case 1: return launch_forward<1>(P, ckpt, sms, s, ring_ctas);
        case 2: return launch_forward<2>(P, ckpt, sms, s, ring_ctas);
        case 3: return launch_forward<3>(P, ckpt, sms, s, ring_ctas);
        case 4: return launch_forward<4>(P, ckpt, sms, s, ring_ctas);
    }
    return SDTW_ERR_UNSUPPORTED;
}
int dispatch_backward(int d, const Params& P, int sms, cudaStream_t s) {
    switch (d) {
        case 1: return launch_backward<1>(P, sms, s);
        case 2: return launch_backward<2>(P, sms, s);
        case 3: return launch_backward<3>(P, sms, s);
        case 4: return launch_backward<4>(P, sms, s);
    }
    return SDTW_ERR_UNSUPPORTED;
}

template <int D, bool SUB, int FW>
int launch_dtw_t(const DtwParams& P, int sms, cudaStream_t stream, int ring_ctas) {
    const int smem = FW * dtw_smem_floats<D>() * 4;
    auto kernel = dtw_kernel<D, SUB, FW>;
    CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    int occ = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, FW * 32, smem));
    if (occ < 1) return SDTW_ERR_UNSUPPORTED;
    long long want, ctas = (long long)sms * occ;
    if (FW == DTW_RING_WARPS) {                     // ring layout: one unit of FW strips at a time per CTA
        want = (long long)((P.NS + FW - 1) / FW) * P.N;
        ctas = std::min(ctas, (long long)ring_ctas);
    } else {
        want = ((long long)P.num_items + FW - 1) / FW;
    }
    const int grid = (int)std::max(1LL, std::min(want, ctas));
    kernel<<<grid, FW * 32, smem, stream>>>(P);
    ++g_launches;
    CUDA_TRY(cudaGetLastError());
    return SDTW_OK;
}
template <int D, bool SUB>
int launch_dtw(const DtwParams& P, int sms, cudaStream_t stream, int ring_ctas) {
    if constexpr (D <= 2) { if (P.ring) return launch_dtw_t<D, SUB, DTW_RING_WARPS>(P, sms, stream, ring_ctas); }
    return launch_dtw_t<D, SUB, DTW_WARPS>(P, sms, stream, 0);
}
template <bool SUB>
int dispatch_dtw(int d, const DtwParams& P, int sms, cudaStream_t s, int ring_ctas) {
    switch (d) {
        case 1: return launch_dtw<1, SUB>(P, sms, s, ring_ctas);
        case 2: return launch_dtw<2, SUB>(P, sms, s, ring_ctas);
        case 3: return launch_dtw<3, SUB>(P, sms, s, ring_ctas);
        case 4: return launch_dtw<4, SUB>(P, sms, s, ring_ctas);
        case 5: return launch_dtw<5, SUB>(P, sms, s, ring_ctas);
        case 6: return launch_dtw<6, SUB>(P, sms, s, ring_ctas);
        case 7: return launch_dtw<7, SUB>(P, sms, s, ring_ctas);
        case 8: return launch_dtw<8, SUB>(P, sms, s, ring_ctas);
        case 9: return launch_dtw<9, SUB>(P, sms, s, ring_ctas);
    }
    return SDTW_ERR_UNSUPPORTED;
}

bool finite_pos(float g) { return std::isfinite(g) && g > 0.f; }

// one evaluation: values (+ gradient) at Z.  If Z_update != nullptr the descent step is fused into the reduction.
int evaluate(const Plan& pl, char* ws, const DeviceInfo& di, const float* Z, const float* X, float gamma, int band,
             float* out_values, float* out_objective, float* out_grad, float* Z_update, float step, cudaStream_t stream,
             int phase = 3, double* out_objective64 = nullptr) {
    // phase bit 0: clears, input scaling, forward sweep, values / objective.  bit 1: reverse sweep, reduction over
    // pairs (+ descent step).  The line search runs the two halves separately (a rejected trial needs no reverse pass).
    const Layout& L = pl.L;
    Params P{};
    float* Xs = reinterpret_cast<float*>(ws + L.off_Xs);
    float* Zs = reinterpret_cast<float*>(ws + L.off_Zs);
    P.Zs = Zs; P.Xs = Xs; P.pm = pl.d_pm;
    P.counters = reinterpret_cast<unsigned*>(ws + L.off_counters);
    P.prog_b = reinterpret_cast<unsigned*>(ws + L.off_prog_b);
    P.hint_b = reinterpret_cast<unsigned*>(ws + L.off_hint_b);
    P.ready_b = reinterpret_cast<unsigned*>(ws + L.off_ready_b);
    P.ring = L.ring_units ? reinterpret_cast<unsigned long long*>(ws + L.off_ring) : nullptr;
    P.ring_prog = L.ring_units ? reinterpret_cast<unsigned*>(ws + L.off_ring_prog) : nullptr;
    P.VP = reinterpret_cast<double*>(ws + L.off_VP);
    P.VS = reinterpret_cast<float*>(ws + L.off_VS);
    P.ES = pl.want_grad ? reinterpret_cast<float*>(ws + L.off_ES) : nullptr;
    P.CK = pl.want_grad ? reinterpret_cast<float*>(ws + L.off_CK) : nullptr;
    P.Gk = pl.want_grad ? reinterpret_cast<float*>(ws + L.off_Gk) : nullptr;
    // reverse-pass statistics (two atomics per work item) are collected only while profiling is enabled
    P.stats = g_profile ? reinterpret_cast<unsigned long long*>(ws + L.off_stats) : nullptr;
    P.dense_reverse = g_dense_reverse;
    P.band = band;
    P.wts = pl.d_w;
    g_last_stats = P.stats;
    g_last_stats_gen = g_ws_gen;
    P.m = (int)pl.m; P.N = pl.N; P.NS = L.NS;
    P.num_items = (unsigned)L.items;
    const double kappa = 1.0 / ((double)gamma * std::log(2.0));
    const float sqrtk = (float)std::sqrt(kappa);
    P.gscale = (float)(2.0 / (double)sqrtk);
    // the kernels see gamma only through the rounded sqrtk; undo exactly that scale on the way out
    const double inv_kappa = 1.0 / ((double)sqrtk * (double)sqrtk);

    ProfScope pr;
    CUDA_TRY((cudaError_t)pr.begin(g_profile));
    CUDA_TRY((cudaError_t)pr.mark(0, stream));
    int rc = SDTW_OK;
    if (phase & 1) {
    {
        // one launch: counters / progress words / rings := 0, strip-boundary columns VS := the sentinel pattern the
        // consumers poll for (sdtw_kernels.cuh), scaled copies of the inputs
        const FillJob f0{reinterpret_cast<uint4*>(ws + L.off_counters), L.sync_bytes / 16, 0u};
        const FillJob f1{reinterpret_cast<uint4*>(ws + L.off_VS), L.vs_bytes / 16, SENTINEL};
        const FillJob f2{reinterpret_cast<uint4*>(ws + L.off_VS), 0, SENTINEL};   // (ES is preset by the forward kernel, strip by strip)
        const long long nx = (long long)pl.offsets[pl.N] * pl.d, nz = (long long)pl.m * pl.d;
        const unsigned long long work = (unsigned long long)(nx + nz) + f0.count16 + f1.count16 + f2.count16;
        const int blocks = (int)std::min<unsigned long long>((work + 255) / 256, (unsigned long long)di.sms * 16);
        prologue_kernel<<<std::max(blocks, 1), 256, 0, stream>>>(f0, f1, f2, X, nx, Z, nz, sqrtk, Xs, Zs);
        ++g_launches;
        CUDA_TRY(cudaGetLastError());
    }
    CUDA_TRY((cudaError_t)pr.mark(1, stream));
    rc = dispatch_forward(pl.d, P, pl.want_grad, di.sms, stream, L.ring_ctas);
    if (rc) return rc;
    } else CUDA_TRY((cudaError_t)pr.mark(1, stream));
    CUDA_TRY((cudaError_t)pr.mark(2, stream));
    if (pl.want_grad && (phase & 2)) {
        rc = dispatch_backward(pl.d, P, di.sms, stream);
        if (rc) return rc;
    }
    CUDA_TRY((cudaError_t)pr.mark(3, stream));
    {
        const int want_values = ((phase & 1) && (out_values || out_objective || out_objective64)) ? 1 : 0;
        const long long md = (pl.want_grad && (phase & 2)) ? (long long)pl.m * pl.d : 0;
        const int blocks = (int)((md + 255) / 256) + want_values;
        if (blocks > 0) {
            epilogue_kernel<<<blocks, 256, 0, stream>>>(P.VP, pl.d_pm, P.wts, pl.N, L.NS, inv_kappa, want_values, out_values,
                                                        out_objective, out_objective64, P.Gk, md, out_grad, Z_update, step);
            ++g_launches;
            CUDA_TRY(cudaGetLastError());
        }
    }
    CUDA_TRY((cudaError_t)pr.mark(4, stream));
    pr.keep();
    return SDTW_OK;
}

int check_common(const void* Z, int64_t m, int32_t d, const void* X, const int64_t* offsets, int32_t N, float gamma,
                 int max_d = SDTW_MAX_D) {
    if (!Z || !X || !offsets || m < 1 || d < 1 || N < 1 || !finite_pos(gamma)) return SDTW_ERR_INVALID_ARG;
    if (offsets[0] != 0) return SDTW_ERR_INVALID_ARG;
    for (int k = 0; k < N; ++k)
        if (offsets[k + 1] <= offsets[k]) return SDTW_ERR_INVALID_ARG;
    if (d > max_d) return SDTW_ERR_UNSUPPORTED;
    return SDTW_OK;
}

// Extended arguments (eq. 7 weights, Table 1 band).  *band_eff: -1 when the band excludes no cell of any pair.
int check_ex(int64_t m, const int64_t* offsets, int32_t N, const float* weights, int64_t band, int* band_eff) {
    if (weights)
        for (int k = 0; k < N; ++k)
            if (!std::isfinite(weights[k])) return SDTW_ERR_INVALID_ARG;
    *band_eff = -1;
    if (band < 0) return SDTW_OK;
    bool excludes = false, narrow = false;
    for (int k = 0; k < N; ++k) {
        const int64_t n = offsets[k + 1] - offsets[k];
        const int64_t gap = n > m ? n - m : m - n;
        if (band < gap) return SDTW_ERR_INVALID_ARG;          // no complete alignment path inside the band
        if (band >= std::max(n, m) - 1) continue;             // every cell of this pair is admissible
        excludes = true;
        // the value staircase (sdtw_kernels.cuh) strays at most W columns / W ceil(n/m) rows from the line
        // i = j n / m, which itself stays within |i - j| <= |n - m|
        const int64_t need = gap + (int64_t)W * ((n + m - 1) / m + 2) + 2;
        if (band < need) narrow = true;
    }
    if (narrow) return SDTW_ERR_UNSUPPORTED;
    if (excludes) *band_eff = (int)std::min<int64_t>(band, (1LL << 30));
    return SDTW_OK;
}

// Workspace: the caller's registered buffer, else a grow-only buffer owned by the library (one per device).  Calls
// are serialised on the buffer by an event: a call on another stream waits for the previous call's work.
struct WsCache { char* ptr = nullptr; size_t bytes = 0; cudaEvent_t last_use = nullptr; };
WsCache g_ws_cache[64];

struct Workspace {
    char* ptr = nullptr;
    WsCache* cache = nullptr;
    cudaStream_t stream = nullptr;
    int acquire(size_t bytes, int dev, cudaStream_t s) {
        stream = s;
        cache = &g_ws_cache[dev];
        if (!cache->last_use) CUDA_TRY(cudaEventCreateWithFlags(&cache->last_use, cudaEventDisableTiming));
        else CUDA_TRY(cudaStreamWaitEvent(s, cache->last_use, 0));
        if (g_user_ws[dev].ptr) {
            if (g_user_ws[dev].bytes < bytes) return SDTW_ERR_WORKSPACE;
            ptr = static_cast<char*>(g_user_ws[dev].ptr);
            return SDTW_OK;
        }
        if (cache->bytes < bytes) {
            if (cache->ptr) {                       // rare: the problem grew; wait for earlier users, then regrow
                CUDA_TRY(cudaEventSynchronize(cache->last_use));
                CUDA_TRY(cudaFree(cache->ptr));
                ++g_ws_gen;
                cache->ptr = nullptr; cache->bytes = 0;
            }
            void* q = nullptr;
            CUDA_TRY(cudaMalloc(&q, bytes));
            cache->ptr = static_cast<char*>(q);
            cache->bytes = bytes;
        }
        ptr = cache->ptr;
        return SDTW_OK;
    }
    ~Workspace() { if (cache && cache->last_use) cudaEventRecord(cache->last_use, stream); }
};

// Small problems are launch-bound: the whole call (all iterations) is captured once on a private stream into a CUDA
// graph, cached on the plan, and replayed on the caller's stream.  Not used while profiling or when a tuning switch of
// sdtw_debug.h is set (the captured launches would bake it in).  `enqueue(stream)` issues the call's launches.
constexpr long long GRAPH_MAX_CELLS = 250000000LL;   // about 1 ms of kernel time per evaluation
cudaStream_t g_capture_stream[64];

bool graph_eligible(const Plan& pl) {
    return pl.cells <= GRAPH_MAX_CELLS && !g_profile && !g_dense_reverse && g_unit_strips == 0 && g_tail_strips < 0 &&
           g_tail_unit == 0 && g_reverse_kernel < 0;
}

template <typename F>
int run_graphed(Plan& pl, const GraphKey& key, cudaStream_t stream, F enqueue) {
    for (auto& ge : pl.graphs) {
        if (ge.key == key) {
            ge.stamp = ++g_stamp;
            CUDA_TRY(cudaGraphLaunch(ge.exec, stream));
            g_launches += ge.launches;
            return SDTW_OK;
        }
    }
    if (std::find(pl.seen.begin(), pl.seen.end(), key) == pl.seen.end()) {   // first time: plain launches
        if (pl.seen.size() >= 8) pl.seen.erase(pl.seen.begin());
        pl.seen.push_back(key);
        return enqueue(stream);
    }
    cudaStream_t& cap = g_capture_stream[pl.dev];
    if (!cap) CUDA_TRY(cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
    const uint64_t launches0 = g_launches;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    int rc = SDTW_OK;
    if (cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return enqueue(stream); }
    rc = enqueue(cap);
    const cudaError_t e_end = cudaStreamEndCapture(cap, &graph);
    const uint64_t n_launch = g_launches - launches0;
    g_launches = launches0;                       // nothing ran during the capture
    if (rc != SDTW_OK || e_end != cudaSuccess || !graph || cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        return rc != SDTW_OK ? rc : enqueue(stream);   // argument errors surface as they would without a graph
    }
    cudaGraphDestroy(graph);
    if (pl.graphs.size() >= 4) {                  // evict the least recently used graph of this plan
        auto it = std::min_element(pl.graphs.begin(), pl.graphs.end(), [](const GraphEntry& a, const GraphEntry& b) { return a.stamp < b.stamp; });
        cudaGraphExecDestroy(it->exec);
        pl.graphs.erase(it);
    }
    GraphEntry ge;
    ge.key = key; ge.exec = exec; ge.launches = n_launch; ge.stamp = ++g_stamp;
    pl.graphs.push_back(ge);
    CUDA_TRY(cudaGraphLaunch(exec, stream));
    g_launches += n_launch;
    return SDTW_OK;
}

// ---- waves: a call whose workspace would not fit is evaluated as consecutive sub-batches of pairs ------------------
// Pairs are independent, so the pair set can be cut into WAVES [b_w, b_{w+1}) of consecutive pairs, each
// evaluated by itself in the same workspace; values land in their slots, the gradients of the waves are added in wave
// order (the sum over pairs is then grouped by wave: a difference of float32 round-off against the unsplit call).
// The budget: sdtw_set_workspace_limit, else the registered workspace, else what the device has free.
__global__ void add_inplace_kernel(float* __restrict__ acc, const float* __restrict__ x, long long count) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < count) acc[e] += x[e];
}
__global__ void sum_objective_kernel(const double* __restrict__ parts, int W, float* __restrict__ out) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < W; ++w) s += parts[w];
        *out = (float)s;
    }
}

size_t workspace_budget(int dev, size_t need) {
    if (g_ws_limit) return g_ws_limit;
    if (g_user_ws[dev].ptr) return g_user_ws[dev].bytes;
    if (g_ws_cache[dev].bytes >= need) return need;
    size_t free_b = 0, total_b = 0;
    if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) { cudaGetLastError(); return need; }
    const size_t avail = free_b + g_ws_cache[dev].bytes;        // the grow-only buffer is freed before it is regrown
    return need <= avail - avail / 16 ? need : avail - avail / 8;
}

// bounds of the waves (bounds[0] = 0 < ... < bounds[W] = N) such that every wave's layout fits `budget`; *max_bytes =
// the largest of them.  SDTW_ERR_WORKSPACE if a single pair does not fit.
int plan_waves(int64_t m, int32_t d, const int64_t* offsets, int32_t N, bool want_grad, int ring_sms, size_t budget,
               std::vector<int>& bounds, size_t* max_bytes, int vs_words = 1) {
    // the split of the last problem is remembered (a descent loop asks for the same one every iteration; under g_mutex)
    struct Memo { int64_t m = 0; int32_t d = 0, N = 0; bool want_grad = false; int ring_sms = 0, vs_words = 0; size_t budget = 0, max_bytes = 0;
                  std::vector<int64_t> offsets; std::vector<int> bounds; };
    static Memo memo;
    if (memo.N == N && memo.m == m && memo.d == d && memo.want_grad == want_grad && memo.ring_sms == ring_sms &&
        memo.vs_words == vs_words && memo.budget == budget && std::memcmp(memo.offsets.data(), offsets, sizeof(int64_t) * (size_t)(N + 1)) == 0) {
        bounds = memo.bounds;
        *max_bytes = memo.max_bytes;
        return SDTW_OK;
    }
    std::vector<int64_t> sub;
    std::vector<int> candidates;                    // wave counts tried: 1 .. 8, then growing by a quarter, at last N
    for (int W = 1; W < N; W = (W < 8 ? W + 1 : W + W / 4)) candidates.push_back(W);
    candidates.push_back(N);
    for (const int W : candidates) {
        bounds.clear();
        for (int w = 0; w <= W; ++w) bounds.push_back((int)((long long)w * N / W));
        size_t mx = 0;
        bool ok = true;
        for (int w = 0; w < W && ok; ++w) {
            const int k0 = bounds[w], k1 = bounds[w + 1];
            sub.assign(offsets + k0, offsets + k1 + 1);
            for (auto& o : sub) o -= offsets[k0];
            Layout L;
            const int rc = build_layout(m, d, sub.data(), k1 - k0, want_grad, L, vs_words, ring_sms);
            if (rc != SDTW_OK) return rc;
            mx = std::max(mx, L.total);
            ok = L.total <= budget;
        }
        if (ok) {
            *max_bytes = mx;
            memo.m = m; memo.d = d; memo.N = N; memo.want_grad = want_grad; memo.ring_sms = ring_sms; memo.vs_words = vs_words; memo.budget = budget;
            memo.max_bytes = mx; memo.offsets.assign(offsets, offsets + N + 1); memo.bounds = bounds;
            return SDTW_OK;
        }
    }
    return SDTW_ERR_WORKSPACE;
}

// one evaluation over waves.  G (m d floats) receives the summed gradient when want_grad; Gtmp is scratch of the same size;
// obj64 (W doubles) scratch for the objective.  out_objective may be null.
int evaluate_waves(const DeviceInfo& di, const std::vector<int>& bounds, char* ws, const float* Z, int64_t m, int32_t d,
                   const float* X, const int64_t* offsets, const float* weights, float gamma, int band_eff, int ring_ok,
                   float* out_values, float* out_objective, float* G, float* Gtmp, double* obj64, cudaStream_t stream) {
    const int W = (int)bounds.size() - 1;
    const long long md = (long long)m * d;
    // every wave has a sub-plan: keep them all cached, or each wave of each iteration would miss (allocation, upload and
    // an eviction whose cudaFree synchronises the device)
    g_plan_cap = std::max(g_plan_cap, (size_t)W + 16);
    g_last_waves = W;
    std::vector<int64_t> sub;
    for (int w = 0; w < W; ++w) {
        const int k0 = bounds[w], k1 = bounds[w + 1];
        sub.assign(offsets + k0, offsets + k1 + 1);
        for (auto& o : sub) o -= offsets[k0];
        Plan* pl = nullptr;
        int rc = get_plan(di, m, d, sub.data(), k1 - k0, weights ? weights + k0 : nullptr, G != nullptr, stream, &pl, 1, ring_ok);
        if (rc) return rc;
        float* Gw = (w == 0) ? G : Gtmp;
        rc = evaluate(*pl, ws, di, Z, X + offsets[k0] * d, gamma, band_eff, out_values ? out_values + k0 : nullptr, nullptr, Gw,
                      nullptr, 0.f, stream, 3, obj64 + w);
        if (rc) return rc;
        if (w > 0 && G) {
            add_inplace_kernel<<<(int)((md + 255) / 256), 256, 0, stream>>>(G, Gtmp, md);
            ++g_launches;
            CUDA_TRY(cudaGetLastError());
        }
    }
    if (out_objective) {
        sum_objective_kernel<<<1, 32, 0, stream>>>(obj64, W, out_objective);
        ++g_launches;
        CUDA_TRY(cudaGetLastError());
    }
    return SDTW_OK;
}

struct DevBuf {
    void* p = nullptr;
    cudaStream_t s = nullptr;
    int alloc(size_t bytes, cudaStream_t st) { s = st; CUDA_TRY(cudaMallocAsync(&p, bytes, st)); return SDTW_OK; }
    ~DevBuf() { if (p) cudaFreeAsync(p, s); }
};

}  // namespace

// =================================================================================================================
extern "C" {

int sdtw_value_grad_ex(const float* Z, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                       float gamma, const float* weights, int64_t band, float* out_values, float* out_grad,
                       float* out_objective, void* stream_) {
    int rc = check_common(Z, m, d, X_concat, offsets, N, gamma);
    if (rc) return rc;
    int band_eff = -1;
    rc = check_ex(m, offsets, N, weights, band, &band_eff);
    if (rc) return rc;
    std::lock_guard<std::mutex> lock(g_mutex);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    DeviceInfo di;
    rc = get_device(di);
    if (rc) return rc;
    const int ring_ok = (out_grad == nullptr && band_eff < 0) ? g_forward_rings : 0;
    const int ring_arg = ring_ok == 2 ? -di.sms : (ring_ok ? di.sms : 0);
    g_last_waves = 1;
    {   // does the workspace of the whole pair set fit?  If not: waves of pairs.  (A cached plan knows the size; only a
        // new shape pays for a layout here.)
        size_t total = 0;
        if (const Plan* hit = find_plan(di.dev, m, d, offsets, N, weights, out_grad != nullptr, 1, ring_ok)) total = hit->L.total;
        else {
            Layout L;
            rc = build_layout(m, d, offsets, N, out_grad != nullptr, L, 1, ring_arg);
            if (rc) return rc;
            total = L.total;
        }
        const size_t budget = workspace_budget(di.dev, total);
        if (total > budget) {
            std::vector<int> bounds;
            size_t max_bytes = 0;
            rc = plan_waves(m, d, offsets, N, out_grad != nullptr, ring_arg, budget, bounds, &max_bytes);
            if (rc) return rc;
            Workspace ws;
            rc = ws.acquire(max_bytes, di.dev, stream);
            if (rc) return rc;
            DevBuf Gtmp, obj64;
            if (out_grad && (rc = Gtmp.alloc((size_t)m * d * 4, stream))) return rc;
            if ((rc = obj64.alloc(sizeof(double) * (bounds.size() - 1), stream))) return rc;
            return evaluate_waves(di, bounds, ws.ptr, Z, m, d, X_concat, offsets, weights, gamma, band_eff, ring_ok, out_values,
                                  out_objective, out_grad, (float*)Gtmp.p, (double*)obj64.p, stream);
        }
    }
    Plan* pl = nullptr;
    rc = get_plan(di, m, d, offsets, N, weights, out_grad != nullptr, stream, &pl, 1, ring_ok);
    if (rc) return rc;
    Workspace ws;
    rc = ws.acquire(pl->L.total, di.dev, stream);
    if (rc) return rc;
    auto enqueue = [&](cudaStream_t st) {
        return evaluate(*pl, ws.ptr, di, Z, X_concat, gamma, band_eff, out_values, out_objective, out_grad, nullptr, 0.f, st);
    };
    if (!graph_eligible(*pl)) return enqueue(stream);
    GraphKey key;
    std::memset(&key, 0, sizeof(key));                 // keys are compared bytewise, padding included
    key.Z = Z; key.X = X_concat; key.values = out_values; key.objective = out_objective; key.grad = out_grad; key.ws = ws.ptr;
    key.iters = -1; key.band = band_eff; key.gamma = gamma; key.step = 0.f;
    return run_graphed(*pl, key, stream, enqueue);
}

int sdtw_value_grad(const float* Z, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                    float gamma, float* out_values, float* out_grad, void* stream_) {
    return sdtw_value_grad_ex(Z, m, d, X_concat, offsets, N, gamma, nullptr, -1, out_values, out_grad, nullptr, stream_);
}

int sdtw_barycenter_ex(float* Z_inout, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                       float gamma, const float* weights, int64_t band, int32_t iters, float step, float* out_values,
                       float* out_objective, void* stream_) {
    int rc = check_common(Z_inout, m, d, X_concat, offsets, N, gamma);
    if (rc) return rc;
    if (iters < 0 || !std::isfinite(step)) return SDTW_ERR_INVALID_ARG;
    int band_eff = -1;
    rc = check_ex(m, offsets, N, weights, band, &band_eff);
    if (rc) return rc;
    std::lock_guard<std::mutex> lock(g_mutex);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    DeviceInfo di;
    rc = get_device(di);
    if (rc) return rc;
    if (iters == 0) return SDTW_OK;
    g_last_waves = 1;
    {   // waves of pairs when the workspace of the whole pair set does not fit (see evaluate_waves)
        size_t total = 0;
        if (const Plan* hit = find_plan(di.dev, m, d, offsets, N, weights, true, 1, 0)) total = hit->L.total;
        else {
            Layout L;
            rc = build_layout(m, d, offsets, N, true, L);
            if (rc) return rc;
            total = L.total;
        }
        const size_t budget = workspace_budget(di.dev, total);
        if (total > budget) {
            std::vector<int> bounds;
            size_t max_bytes = 0;
            rc = plan_waves(m, d, offsets, N, true, 0, budget, bounds, &max_bytes);
            if (rc) return rc;
            Workspace ws;
            rc = ws.acquire(max_bytes, di.dev, stream);
            if (rc) return rc;
            DevBuf G, Gtmp, obj64;
            const long long md = (long long)m * d;
            if ((rc = G.alloc((size_t)md * 4, stream)) || (rc = Gtmp.alloc((size_t)md * 4, stream)) ||
                (rc = obj64.alloc(sizeof(double) * (bounds.size() - 1), stream)))
                return rc;
            for (int it = 0; it < iters; ++it) {
                rc = evaluate_waves(di, bounds, ws.ptr, Z_inout, m, d, X_concat, offsets, weights, gamma, band_eff, false,
                                    it == iters - 1 ? out_values : nullptr, out_objective ? out_objective + it : nullptr,
                                    (float*)G.p, (float*)Gtmp.p, (double*)obj64.p, stream);
                if (rc) return rc;
                gd_update_kernel<<<(int)((md + 255) / 256), 256, 0, stream>>>(Z_inout, (const float*)G.p, md, step);
                ++g_launches;
                CUDA_TRY(cudaGetLastError());
            }
            return SDTW_OK;
        }
    }
    Plan* pl = nullptr;
    rc = get_plan(di, m, d, offsets, N, weights, true, stream, &pl);
    if (rc) return rc;
    Workspace ws;
    rc = ws.acquire(pl->L.total, di.dev, stream);
    if (rc) return rc;
    auto enqueue = [&](cudaStream_t st) {
        for (int it = 0; it < iters; ++it) {
            float* vals = (it == iters - 1) ? out_values : nullptr;
            float* obj = out_objective ? out_objective + it : nullptr;
            const int r = evaluate(*pl, ws.ptr, di, Z_inout, X_concat, gamma, band_eff, vals, obj, nullptr, Z_inout, step, st);
            if (r) return r;
        }
        return (int)SDTW_OK;
    };
    if (!graph_eligible(*pl)) return enqueue(stream);
    GraphKey key;
    std::memset(&key, 0, sizeof(key));
    key.Z = Z_inout; key.X = X_concat; key.values = out_values; key.objective = out_objective; key.grad = nullptr; key.ws = ws.ptr;
    key.iters = iters; key.band = band_eff; key.gamma = gamma; key.step = step;
    return run_graphed(*pl, key, stream, enqueue);
}

int sdtw_barycenter_backtracking(float* Z_inout, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets,
                                 int32_t N, float gamma, const float* weights, int64_t band, int32_t iters, float step0,
                                 float shrink, float c1, int32_t max_trials, float* out_values, double* out_objective,
                                 float* out_steps, int32_t* out_trials, void* stream_) {
    int rc = check_common(Z_inout, m, d, X_concat, offsets, N, gamma);
    if (rc) return rc;
    if (iters < 0 || !(std::isfinite(step0) && step0 > 0.f) || !(shrink > 0.f && shrink < 1.f) ||
        !(std::isfinite(c1) && c1 >= 0.f) || max_trials < 1 || !out_objective || (iters > 0 && (!out_steps || !out_trials)))
        return SDTW_ERR_INVALID_ARG;
    int band_eff = -1;
    rc = check_ex(m, offsets, N, weights, band, &band_eff);
    if (rc) return rc;
    std::lock_guard<std::mutex> lock(g_mutex);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    DeviceInfo di;
    rc = get_device(di);
    if (rc) return rc;
    Plan* pl = nullptr;
    rc = get_plan(di, m, d, offsets, N, weights, true, stream, &pl);
    if (rc) return rc;
    Workspace ws;
    rc = ws.acquire(pl->L.total, di.dev, stream);
    if (rc) return rc;
    const Layout& L = pl->L;
    float* G = reinterpret_cast<float*>(ws.ptr + L.off_G);
    float* Zt = reinterpret_cast<float*>(ws.ptr + L.off_Zt);
    float* Vt = reinterpret_cast<float*>(ws.ptr + L.off_Vt);
    double* scal = reinterpret_cast<double*>(ws.ptr + L.off_scal);      // [0] objective, [1] ||G||^2
    const long long md = (long long)m * d;
    const int blocks = (int)((md + 255) / 256);
    double h[2] = {0.0, 0.0};
    auto read_scalars = [&]() -> int {
        CUDA_TRY(cudaMemcpyAsync(h, scal, sizeof(h), cudaMemcpyDeviceToHost, stream));
        CUDA_TRY(cudaStreamSynchronize(stream));
        return SDTW_OK;
    };
    auto gradient_norm = [&]() -> int {
        sqnorm_kernel<<<1, 1024, 0, stream>>>(G, md, scal + 1);
        ++g_launches;
        CUDA_TRY(cudaGetLastError());
        return SDTW_OK;
    };
    // f, values and G at Z0
    rc = evaluate(*pl, ws.ptr, di, Z_inout, X_concat, gamma, band_eff, out_values, nullptr, G, nullptr, 0.f, stream, 3, scal);
    if (rc || (rc = gradient_norm()) || (rc = read_scalars())) return rc;
    double f = h[0], gg = h[1];
    out_objective[0] = f;
    bool stopped = false;
    for (int it = 0; it < iters; ++it) {
        out_steps[it] = 0.f; out_trials[it] = 0;
        if (!stopped) {
            double t = step0;
            bool accepted = false;
            for (int tr = 0; tr < max_trials; ++tr) {
                trial_point_kernel<<<blocks, 256, 0, stream>>>(Zt, Z_inout, G, md, (float)t);
                ++g_launches;
                CUDA_TRY(cudaGetLastError());
                // forward sweep only (with checkpoints: an accepted trial goes straight on to its reverse sweep)
                rc = evaluate(*pl, ws.ptr, di, Zt, X_concat, gamma, band_eff, Vt, nullptr, nullptr, nullptr, 0.f, stream, 1, scal);
                if (rc || (rc = read_scalars())) return rc;
                out_trials[it] = tr + 1;
                if (h[0] <= f - (double)c1 * t * gg) {                 // Armijo condition, on the host in double
                    CUDA_TRY(cudaMemcpyAsync(Z_inout, Zt, (size_t)md * 4, cudaMemcpyDeviceToDevice, stream));
                    if (out_values) CUDA_TRY(cudaMemcpyAsync(out_values, Vt, (size_t)N * 4, cudaMemcpyDeviceToDevice, stream));
                    rc = evaluate(*pl, ws.ptr, di, Zt, X_concat, gamma, band_eff, nullptr, nullptr, G, nullptr, 0.f, stream, 2);
                    if (rc || (rc = gradient_norm()) || (rc = read_scalars())) return rc;
                    f = h[0]; gg = h[1];
                    out_steps[it] = (float)t;
                    accepted = true;
                    break;
                }
                t *= (double)shrink;
            }
            if (!accepted) stopped = true;
        }
        out_objective[it + 1] = f;
    }
    return SDTW_OK;
}

int sdtw_barycenter_lbfgs(float* Z_inout, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                          float gamma, const float* weights, int64_t band, int32_t iters, int32_t hist, float step0,
                          float shrink, float c1, int32_t max_trials, float* out_values, double* out_objective,
                          float* out_steps, int32_t* out_trials, void* stream_) {
    int rc = check_common(Z_inout, m, d, X_concat, offsets, N, gamma);
    if (rc) return rc;
    if (iters < 0 || hist < 0 || hist > 64 || !(std::isfinite(step0) && step0 > 0.f) || !(shrink > 0.f && shrink < 1.f) ||
        !(std::isfinite(c1) && c1 >= 0.f) || max_trials < 1 || !out_objective || (iters > 0 && (!out_steps || !out_trials)))
        return SDTW_ERR_INVALID_ARG;
    int band_eff = -1;
    rc = check_ex(m, offsets, N, weights, band, &band_eff);
    if (rc) return rc;
    std::lock_guard<std::mutex> lock(g_mutex);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    DeviceInfo di;
    rc = get_device(di);
    if (rc) return rc;
    Plan* pl = nullptr;
    rc = get_plan(di, m, d, offsets, N, weights, true, stream, &pl);
    if (rc) return rc;
    Workspace ws;
    rc = ws.acquire(pl->L.total, di.dev, stream);
    if (rc) return rc;
    const Layout& L = pl->L;
    const long long md = (long long)m * d;
    const int blocks = (int)((md + 255) / 256);
    float* G = reinterpret_cast<float*>(ws.ptr + L.off_G);           // gradient at the current iterate
    float* Zt = reinterpret_cast<float*>(ws.ptr + L.off_Zt);         // trial point
    float* Vt = reinterpret_cast<float*>(ws.ptr + L.off_Vt);
    double* scal = reinterpret_cast<double*>(ws.ptr + L.off_scal);   // [0] objective, [1] dot product
    // direction, the gradient at the accepted point, and the stored pairs (s_i, y_i): stream-ordered scratch
    DevBuf vec;
    const int H = std::max(hist, 1);
    if ((rc = vec.alloc((size_t)(2 + 2 * H) * md * 4, stream))) return rc;
    float* Dv = static_cast<float*>(vec.p);
    float* Gn = Dv + md;
    float* S = Gn + md;                                                // [H][md], slot i
    float* Y = S + (size_t)H * md;
    double h[2] = {0.0, 0.0};
    auto read_scalars = [&]() -> int {
        CUDA_TRY(cudaMemcpyAsync(h, scal, sizeof(h), cudaMemcpyDeviceToHost, stream));
        CUDA_TRY(cudaStreamSynchronize(stream));
        return SDTW_OK;
    };
    auto dot = [&](const float* a, const float* b, double* out) -> int {      // blocks the host: the recursion needs the value
        dot_kernel<<<1, 1024, 0, stream>>>(a, b, md, scal + 1);
        ++g_launches;
        CUDA_TRY(cudaGetLastError());
        int r = read_scalars();
        *out = h[1];
        return r;
    };
    auto axpby = [&](float* y, const float* x, double a, double b) -> int {
        axpby_kernel<<<blocks, 256, 0, stream>>>(y, x, md, (float)a, (float)b);
        ++g_launches;
        CUDA_TRY(cudaGetLastError());
        return SDTW_OK;
    };
    // f, values and G at Z0
    rc = evaluate(*pl, ws.ptr, di, Z_inout, X_concat, gamma, band_eff, out_values, nullptr, G, nullptr, 0.f, stream, 3, scal);
    if (rc || (rc = read_scalars())) return rc;
    double f = h[0];
    out_objective[0] = f;
    std::vector<int> slots;                                            // ring slots of the stored pairs, oldest first
    std::vector<double> rho, alpha;
    bool stopped = false;
    for (int it = 0; it < iters; ++it) {
        out_steps[it] = 0.f; out_trials[it] = 0;
        if (!stopped) {
            // d = -H G: the two-loop recursion over the stored pairs (include/sdtw.h); scalars in float64 on the host
            if ((rc = axpby(Dv, G, 1.0, 0.0))) return rc;             // q = G
            alpha.assign(slots.size(), 0.0);
            for (int i = (int)slots.size() - 1; i >= 0; --i) {
                double sq;
                if ((rc = dot(S + (size_t)slots[i] * md, Dv, &sq))) return rc;
                alpha[i] = rho[i] * sq;
                if ((rc = axpby(Dv, Y + (size_t)slots[i] * md, -alpha[i], 1.0))) return rc;
            }
            if (!slots.empty()) {
                const float* sn = S + (size_t)slots.back() * md; const float* yn = Y + (size_t)slots.back() * md;
                double sy, yy;
                if ((rc = dot(sn, yn, &sy)) || (rc = dot(yn, yn, &yy))) return rc;
                if ((rc = axpby(Dv, Dv, sy / yy, 0.0))) return rc;   // r = (s.y / y.y) q
            }
            for (size_t i = 0; i < slots.size(); ++i) {
                double yr;
                if ((rc = dot(Y + (size_t)slots[i] * md, Dv, &yr))) return rc;
                if ((rc = axpby(Dv, S + (size_t)slots[i] * md, alpha[i] - rho[i] * yr, 1.0))) return rc;
            }
            if ((rc = axpby(Dv, Dv, -1.0, 0.0))) return rc;          // d = -r
            double gd;
            if ((rc = dot(G, Dv, &gd))) return rc;
            if (!(gd < 0.0)) {                                        // not a descent direction: restart from -G
                slots.clear(); rho.clear();
                if ((rc = axpby(Dv, G, -1.0, 0.0)) || (rc = dot(G, Dv, &gd))) return rc;
            }
            double t = slots.empty() ? (double)step0 : 1.0;
            bool accepted = false;
            for (int tr = 0; tr < max_trials; ++tr) {
                trial_point_kernel<<<blocks, 256, 0, stream>>>(Zt, Z_inout, Dv, md, (float)-t);   // Zt = Z - (-t) d = Z + t d
                ++g_launches;
                CUDA_TRY(cudaGetLastError());
                rc = evaluate(*pl, ws.ptr, di, Zt, X_concat, gamma, band_eff, Vt, nullptr, nullptr, nullptr, 0.f, stream, 1, scal);
                if (rc || (rc = read_scalars())) return rc;
                out_trials[it] = tr + 1;
                if (h[0] <= f + (double)c1 * t * gd) {                 // Armijo condition, on the host in double
                    // gradient at the accepted point (reverse sweep on the checkpoints the trial wrote), then the pair
                    rc = evaluate(*pl, ws.ptr, di, Zt, X_concat, gamma, band_eff, nullptr, nullptr, Gn, nullptr, 0.f, stream, 2);
                    if (rc) return rc;
                    f = h[0];
                    if (hist > 0) {
                        int slot;
                        if ((int)slots.size() == hist) { slot = slots.front(); slots.erase(slots.begin()); rho.erase(rho.begin()); }
                        else { slot = 0; while (std::find(slots.begin(), slots.end(), slot) != slots.end()) ++slot; }
                        float* sn = S + (size_t)slot * md; float* yn = Y + (size_t)slot * md;
                        diff_kernel<<<blocks, 256, 0, stream>>>(sn, Zt, Z_inout, md);
                        diff_kernel<<<blocks, 256, 0, stream>>>(yn, Gn, G, md);
                        g_launches += 2;
                        CUDA_TRY(cudaGetLastError());
                        double sy, ss, yy;
                        if ((rc = dot(sn, yn, &sy)) || (rc = dot(sn, sn, &ss)) || (rc = dot(yn, yn, &yy))) return rc;
                        if (sy > 1e-10 * std::sqrt(ss) * std::sqrt(yy)) { slots.push_back(slot); rho.push_back(1.0 / sy); }
                    }
                    CUDA_TRY(cudaMemcpyAsync(Z_inout, Zt, (size_t)md * 4, cudaMemcpyDeviceToDevice, stream));
                    CUDA_TRY(cudaMemcpyAsync(G, Gn, (size_t)md * 4, cudaMemcpyDeviceToDevice, stream));
                    if (out_values) CUDA_TRY(cudaMemcpyAsync(out_values, Vt, (size_t)N * 4, cudaMemcpyDeviceToDevice, stream));
                    out_steps[it] = (float)t;
                    accepted = true;
                    break;
                }
                t *= (double)shrink;
            }
            if (!accepted) stopped = true;
        }
        out_objective[it + 1] = f;
    }
    return SDTW_OK;
}

int sdtw_barycenter(float* Z_inout, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                    float gamma, int32_t iters, float step, float* out_values, float* out_objective, void* stream_) {
    return sdtw_barycenter_ex(Z_inout, m, d, X_concat, offsets, N, gamma, nullptr, -1, iters, step, out_values,
                              out_objective, stream_);
}

// one launch of the DTW / Sub-DTW kernel over the pairs of `offsets` (a whole call, or one wave of it) in workspace `wsp`
static int dtw_launch(bool sub, const DeviceInfo& di, char* wsp, const float* Z, int64_t m, int32_t d, const float* X_concat,
                      const int64_t* offsets, int32_t N, float* out_val, int32_t* out_i0, float* out_score, int32_t* out_i1,
                      cudaStream_t stream);

static int dtw_common(bool sub, const float* Z, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets,
                      int32_t N, float* out_val, int32_t* out_i0, float* out_score, int32_t* out_i1, void* stream_) {
    int rc = check_common(Z, m, d, X_concat, offsets, N, 1.0f, SDTW_DTW_MAX_D);
    if (rc) return rc;
    for (int k = 0; k < N; ++k)          // path lengths / start rows are carried as floats, exact below 2^24
        if (offsets[k + 1] - offsets[k] + m >= (1LL << 24)) return SDTW_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_mutex);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    DeviceInfo di;
    rc = get_device(di);
    if (rc) return rc;
    // WAVES (sdtw.h): pairs are independent and every output is per pair, so a pair set whose boundary state exceeds the
    // budget is swept as consecutive waves of pairs in the same workspace; every output bit is that of the unsplit call
    size_t total = 0;
    const int ring_arg = g_forward_rings == 2 ? -di.sms : (g_forward_rings ? di.sms : 0);
    if (const Plan* hit = find_plan(di.dev, m, d, offsets, N, nullptr, false, 2, g_forward_rings)) total = hit->L.total;
    else {
        Layout L0;
        rc = build_layout(m, d, offsets, N, false, L0, 2, ring_arg);
        if (rc) return rc;
        total = L0.total;
    }
    g_last_waves = 1;
    const size_t budget = workspace_budget(di.dev, total);
    if (total <= budget) {
        Workspace ws;
        rc = ws.acquire(total, di.dev, stream);
        if (rc) return rc;
        return dtw_launch(sub, di, ws.ptr, Z, m, d, X_concat, offsets, N, out_val, out_i0, out_score, out_i1, stream);
    }
    std::vector<int> bounds;
    size_t max_bytes = 0;
    rc = plan_waves(m, d, offsets, N, false, ring_arg, budget, bounds, &max_bytes, 2);
    if (rc) return rc;
    Workspace ws;
    rc = ws.acquire(max_bytes, di.dev, stream);
    if (rc) return rc;
    const int W = (int)bounds.size() - 1;
    g_plan_cap = std::max(g_plan_cap, (size_t)W + 16);
    g_last_waves = W;
    std::vector<int64_t> subo;
    for (int w = 0; w < W; ++w) {
        const int k0 = bounds[w], k1 = bounds[w + 1];
        subo.assign(offsets + k0, offsets + k1 + 1);
        for (auto& o : subo) o -= offsets[k0];
        rc = dtw_launch(sub, di, ws.ptr, Z, m, d, X_concat + offsets[k0] * d, subo.data(), k1 - k0, out_val ? out_val + k0 : nullptr,
                        out_i0 ? out_i0 + k0 : nullptr, out_score ? out_score + k0 : nullptr, out_i1 ? out_i1 + k0 : nullptr, stream);
        if (rc) return rc;
    }
    return SDTW_OK;
}

static int dtw_launch(bool sub, const DeviceInfo& di, char* wsp, const float* Z, int64_t m, int32_t d, const float* X_concat,
                      const int64_t* offsets, int32_t N, float* out_val, int32_t* out_i0, float* out_score, int32_t* out_i1,
                      cudaStream_t stream) {
    Plan* pl = nullptr;
    int rc = get_plan(di, m, d, offsets, N, nullptr, false, stream, &pl, 2, g_forward_rings);
    if (rc) return rc;
    struct { char* ptr; } ws{wsp};
    const Layout& L = pl->L;
    DtwParams P{};
    P.Z = Z; P.X = X_concat; P.pm = pl->d_pm;
    P.counter = reinterpret_cast<unsigned*>(ws.ptr + L.off_counters);
    P.VS = reinterpret_cast<unsigned*>(ws.ptr + L.off_VS);
    P.ring = L.ring_units ? reinterpret_cast<unsigned long long*>(ws.ptr + L.off_ring) : nullptr;
    P.ring_prog = L.ring_units ? reinterpret_cast<unsigned*>(ws.ptr + L.off_ring_prog) : nullptr;
    P.out_dtw = out_val; P.out_len = out_i0; P.out_score = out_score; P.out_b = out_i1;
    P.m = (int)m; P.N = N; P.NS = L.NS; P.num_items = (unsigned)L.items;
    ProfScope pr;
    CUDA_TRY((cudaError_t)pr.begin(g_profile));
    CUDA_TRY((cudaError_t)pr.mark(0, stream));
    CUDA_TRY(cudaMemsetAsync(ws.ptr + L.off_counters, 0, L.sync_bytes, stream));
    CUDA_TRY(cudaMemsetAsync(ws.ptr + L.off_VS, 0xFF, L.vs_bytes, stream));   // sentinel preset (dtw_kernel.cuh)
    CUDA_TRY((cudaError_t)pr.mark(1, stream));
    rc = sub ? dispatch_dtw<true>(d, P, di.sms, stream, L.ring_ctas) : dispatch_dtw<false>(d, P, di.sms, stream, L.ring_ctas);
    if (rc) return rc;
    for (int i = 2; i <= 4; ++i) CUDA_TRY((cudaError_t)pr.mark(i, stream));   // "forward" slot = the DTW kernel
    pr.keep();
    return SDTW_OK;
}

int sdtw_dtw_score(const float* Z, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                   float* out_dtw, int32_t* out_pathlen, float* out_score, void* stream_) {
    return dtw_common(false, Z, m, d, X_concat, offsets, N, out_dtw, out_pathlen, out_score, nullptr, stream_);
}

int sdtw_subdtw(const float* Z, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                float* out_value, int32_t* out_a, int32_t* out_b, void* stream_) {
    return dtw_common(true, Z, m, d, X_concat, offsets, N, out_value, out_a, nullptr, out_b, stream_);
}

int sdtw_gd_update(float* Z_inout, const float* G, int64_t count, float step, void* stream_) {
    if (!Z_inout || !G || count < 1 || !std::isfinite(step)) return SDTW_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_mutex);
    DeviceInfo di;
    int rc = get_device(di);
    if (rc) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    gd_update_kernel<<<(int)((count + 255) / 256), 256, 0, stream>>>(Z_inout, G, count, step);
    ++g_launches;
    CUDA_TRY(cudaGetLastError());
    return SDTW_OK;
}

// ---- host-buffer variants ---------------------------------------------------------------------------------------

int sdtw_value_grad_host(const float* Z, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                         float gamma, float* out_values, float* out_grad, void* stream_) {
    int rc = check_common(Z, m, d, X_concat, offsets, N, gamma);
    if (rc) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const size_t zb = (size_t)m * d * 4, xb = (size_t)offsets[N] * d * 4;
    DevBuf dZ, dX, dV, dG;
    if ((rc = dZ.alloc(zb, stream)) || (rc = dX.alloc(xb, stream)) || (rc = dV.alloc((size_t)N * 4, stream)) ||
        (rc = dG.alloc(zb, stream)))
        return rc;
    CUDA_TRY(cudaMemcpyAsync(dZ.p, Z, zb, cudaMemcpyHostToDevice, stream));
    CUDA_TRY(cudaMemcpyAsync(dX.p, X_concat, xb, cudaMemcpyHostToDevice, stream));
    rc = sdtw_value_grad((const float*)dZ.p, m, d, (const float*)dX.p, offsets, N, gamma, out_values ? (float*)dV.p : nullptr,
                         out_grad ? (float*)dG.p : nullptr, stream_);
    if (rc) return rc;
    if (out_values) CUDA_TRY(cudaMemcpyAsync(out_values, dV.p, (size_t)N * 4, cudaMemcpyDeviceToHost, stream));
    if (out_grad) CUDA_TRY(cudaMemcpyAsync(out_grad, dG.p, zb, cudaMemcpyDeviceToHost, stream));
    CUDA_TRY(cudaStreamSynchronize(stream));
    return SDTW_OK;
}

int sdtw_barycenter_host(float* Z_inout, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                         float gamma, int32_t iters, float step, float* out_values, float* out_objective, void* stream_) {
    int rc = check_common(Z_inout, m, d, X_concat, offsets, N, gamma);
    if (rc) return rc;
    if (iters < 0 || !std::isfinite(step)) return SDTW_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const size_t zb = (size_t)m * d * 4, xb = (size_t)offsets[N] * d * 4;
    DevBuf dZ, dX, dV, dO;
    if ((rc = dZ.alloc(zb, stream)) || (rc = dX.alloc(xb, stream)) || (rc = dV.alloc((size_t)N * 4, stream)) ||
        (rc = dO.alloc((size_t)std::max(iters, 1) * 4, stream)))
        return rc;
    CUDA_TRY(cudaMemcpyAsync(dZ.p, Z_inout, zb, cudaMemcpyHostToDevice, stream));
    CUDA_TRY(cudaMemcpyAsync(dX.p, X_concat, xb, cudaMemcpyHostToDevice, stream));
    rc = sdtw_barycenter((float*)dZ.p, m, d, (const float*)dX.p, offsets, N, gamma, iters, step,
                         out_values ? (float*)dV.p : nullptr, out_objective ? (float*)dO.p : nullptr, stream_);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpyAsync(Z_inout, dZ.p, zb, cudaMemcpyDeviceToHost, stream));
    if (out_values && iters > 0) CUDA_TRY(cudaMemcpyAsync(out_values, dV.p, (size_t)N * 4, cudaMemcpyDeviceToHost, stream));
    if (out_objective && iters > 0) CUDA_TRY(cudaMemcpyAsync(out_objective, dO.p, (size_t)iters * 4, cudaMemcpyDeviceToHost, stream));
    CUDA_TRY(cudaStreamSynchronize(stream));
    return SDTW_OK;
}

// ---- sdtw_value_static: the forward-only sweep with its scratch in a static device array (no allocation) ----------
}  // extern "C"

// The one scratch array of sdtw_value_static (include/sdtw.h).  It belongs to this library's CUDA module: each GPU the
// module is loaded on holds its own copy until the process exits.  In HOST code the name g_static_scratch is only a
// handle of the symbol -- not an address a kernel can use; the device address comes from cudaGetSymbolAddress
// (static_scratch_ptr below).  DEVICE code may name the array directly (static_meta_kernel does).
static __device__ __align__(256) unsigned char g_static_scratch[SDTW_STATIC_SCRATCH_BYTES];

namespace {

// The per-pair schedule table, passed by value as a kernel argument so that no host-to-device copy is needed.
struct StaticMeta { PairMeta pm[SDTW_STATIC_MAX_PAIRS]; };
static_assert(sizeof(StaticMeta) <= 4000, "the schedule table must fit the kernel argument space");

// Writes the schedule table into the scratch array at byte offset `off` (device code: names the array itself).
__global__ void static_meta_kernel(const __grid_constant__ StaticMeta meta, int N, unsigned long long off) {
    PairMeta* dst = reinterpret_cast<PairMeta*>(g_static_scratch + off);
    for (int i = threadIdx.x; i < N; i += blockDim.x) dst[i] = meta.pm[i];
}

// Device address of g_static_scratch on the CURRENT device, resolved once per device (under g_mutex).
int static_scratch_ptr(int dev, char** out) {
    static char* ptr[64] = {};
    if (!ptr[dev]) {
        void* p = nullptr;
        CUDA_TRY(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) return SDTW_ERR_UNSUPPORTED;
        ptr[dev] = static_cast<char*>(p);
    }
    *out = ptr[dev];
    return SDTW_OK;
}

}  // namespace

extern "C" {

int sdtw_value_static(const float* Z, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                      float gamma, float* out_values, void* stream_) {
    int rc = check_common(Z, m, d, X_concat, offsets, N, gamma);
    if (rc) return rc;
    if (!out_values) return SDTW_ERR_INVALID_ARG;
    if (N > SDTW_STATIC_MAX_PAIRS) return SDTW_ERR_STATIC_LIMIT;
    // a Plan that lives on this stack frame only: same layout as sdtw_value_grad(out_grad = NULL) with a boundary column
    // per strip (no rings, so the layout does not depend on the device), the schedule table appended behind it
    Plan pl;
    rc = build_layout(m, d, offsets, N, false, pl.L, 1, 0);
    if (rc) return rc;
    const size_t off_pm = align_up(pl.L.total, 256);
    if (off_pm + sizeof(PairMeta) * (size_t)N > (size_t)SDTW_STATIC_SCRATCH_BYTES) return SDTW_ERR_STATIC_LIMIT;
    std::lock_guard<std::mutex> lock(g_mutex);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    DeviceInfo di;
    rc = get_device(di);
    if (rc) return rc;
    char* scratch = nullptr;
    rc = static_scratch_ptr(di.dev, &scratch);      // first call on this device: cudaGetSymbolAddress
    if (rc) return rc;
    pl.dev = di.dev; pl.m = m; pl.d = d; pl.N = N; pl.want_grad = false;
    pl.offsets.assign(offsets, offsets + N + 1);
    pl.cells = (long long)offsets[N] * m;
    pl.d_pm = reinterpret_cast<PairMeta*>(scratch + off_pm);
    StaticMeta meta;
    std::memset(&meta, 0, sizeof(meta));
    for (int ps = 0; ps < N; ++ps) meta.pm[ps] = pl.L.pm[ps];
    static_meta_kernel<<<1, 64, 0, stream>>>(meta, N, (unsigned long long)off_pm);
    ++g_launches;
    CUDA_TRY(cudaGetLastError());
    // the sweep itself: evaluate() clears the counters and presets the boundary columns in its prologue launch, so the
    // previous call's contents of the array do not matter.  Profiling would create events: off for this call.
    const bool profile = g_profile;
    g_profile = false;
    rc = evaluate(pl, scratch, di, Z, X_concat, gamma, -1, out_values, nullptr, nullptr, nullptr, 0.f, stream);
    g_profile = profile;
    return rc;
}

// ---- workspace, status, instrumentation -------------------------------------------------------------------------
size_t sdtw_workspace_bytes_ex(int64_t m, int32_t d, const int64_t* offsets, int32_t N, int want_grad, int64_t band) {
    Layout L;
    int sms = 148;                                  // the layout of forward-only calls depends on the SM count: B200 unless
    DeviceInfo di;                                  // a device is current
    if (get_device(di) == SDTW_OK) sms = di.sms;
    int band_eff = -1;
    if (band >= 0 && offsets && N >= 1 && m >= 1 && check_ex(m, offsets, N, nullptr, band, &band_eff) != SDTW_OK) return 0;
    const int ring_arg = (!want_grad && band_eff < 0) ? (g_forward_rings == 2 ? -sms : (g_forward_rings ? sms : 0)) : 0;
    if (build_layout(m, d, offsets, N, want_grad != 0, L, 1, ring_arg) != SDTW_OK) return 0;
    return L.total;
}

size_t sdtw_workspace_bytes(int64_t m, int32_t d, const int64_t* offsets, int32_t N, int want_grad) {
    return sdtw_workspace_bytes_ex(m, d, offsets, N, want_grad, -1);
}

size_t sdtw_dtw_workspace_bytes(int64_t m, int32_t d, const int64_t* offsets, int32_t N) {
    Layout L;
    int sms = 148;
    DeviceInfo di;
    if (get_device(di) == SDTW_OK) sms = di.sms;
    if (build_layout(m, d, offsets, N, false, L, 2, g_forward_rings == 2 ? -sms : (g_forward_rings ? sms : 0)) != SDTW_OK) return 0;
    return L.total;
}

int sdtw_set_workspace_limit(size_t bytes) {
    std::lock_guard<std::mutex> lock(g_mutex);
    g_ws_limit = bytes;
    return SDTW_OK;
}

int sdtw_set_workspace(void* dev_ptr, size_t bytes) {
    std::lock_guard<std::mutex> lock(g_mutex);
    if (dev_ptr && (reinterpret_cast<uintptr_t>(dev_ptr) & 255u)) return SDTW_ERR_INVALID_ARG;
    if (!dev_ptr && bytes) return SDTW_ERR_INVALID_ARG;
    int dev = 0;                                    // the registration belongs to the CURRENT device
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return SDTW_ERR_UNSUPPORTED;
    g_user_ws[dev].ptr = dev_ptr;
    g_user_ws[dev].bytes = dev_ptr ? bytes : 0;
    ++g_ws_gen;
    if (!dev_ptr) {                                 // also drop the library-owned buffer of the current device
        if (g_ws_cache[dev].ptr) {
            if (g_ws_cache[dev].last_use) cudaEventSynchronize(g_ws_cache[dev].last_use);
            cudaFree(g_ws_cache[dev].ptr);
            g_ws_cache[dev].ptr = nullptr;
            g_ws_cache[dev].bytes = 0;
        }
    }
    return SDTW_OK;
}

const char* sdtw_status_string(int status) {
    switch (status) {
        case SDTW_OK: return "ok";
        case SDTW_ERR_INVALID_ARG: return "invalid argument";
        case SDTW_ERR_UNSUPPORTED: return "unsupported (d > SDTW_MAX_D, size beyond limits, or device is not sm_100)";
        case SDTW_ERR_WORKSPACE:
            return "workspace budget too small: the registered workspace (or the sdtw_set_workspace_limit / free-memory budget) "
                   "does not hold this call, or, for calls that split into waves, not even one pair";
        case SDTW_ERR_CUDA: return "CUDA runtime error (see sdtw_last_cuda_error)";
        case SDTW_ERR_STATIC_LIMIT:
            return "sdtw_value_static: more than SDTW_STATIC_MAX_PAIRS pairs, or the sweep needs more scratch than the built-in "
                   "SDTW_STATIC_SCRATCH_BYTES array holds (use sdtw_value_grad with a registered workspace instead)";
    }
    return "unknown status";
}

int sdtw_last_cuda_error(void) { return g_last_cuda_error; }

int sdtw_last_wave_count(void) { return g_last_waves; }

uint64_t sdtw_launch_count(void) {
    std::lock_guard<std::mutex> lock(g_mutex);
    return g_launches;
}

int sdtw_profile_enable(int on) {
    std::lock_guard<std::mutex> lock(g_mutex);
    g_profile = on != 0;
    return SDTW_OK;
}

int sdtw_profile_read(double* ms_forward, double* ms_backward, double* ms_other, int64_t* evaluations) {
    std::lock_guard<std::mutex> lock(g_mutex);
    double f = 0, b = 0, o = 0;
    for (auto& pr : g_prof) {
        CUDA_TRY(cudaEventSynchronize(pr.e[4]));
        float t = 0;
        CUDA_TRY(cudaEventElapsedTime(&t, pr.e[1], pr.e[2])); f += t;
        CUDA_TRY(cudaEventElapsedTime(&t, pr.e[2], pr.e[3])); b += t;
        CUDA_TRY(cudaEventElapsedTime(&t, pr.e[0], pr.e[1])); o += t;   // prologue: clears, sentinel preset, input scaling
        CUDA_TRY(cudaEventElapsedTime(&t, pr.e[3], pr.e[4])); o += t;   // values, reduction over pairs, descent step
        for (auto& e : pr.e) cudaEventDestroy(e);
    }
    if (ms_forward) *ms_forward = f;
    if (ms_backward) *ms_backward = b;
    if (ms_other) *ms_other = o;
    if (evaluations) *evaluations = (int64_t)g_prof.size();
    g_prof.clear();
    return SDTW_OK;
}

int sdtw_set_schedule_tail(int tail_strips, int tail_unit) {
    std::lock_guard<std::mutex> lock(g_mutex);
    g_tail_strips = tail_strips;
    g_tail_unit = tail_unit;
    return SDTW_OK;
}

int sdtw_set_schedule(int unit_strips) {
    if (unit_strips < 0) return SDTW_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_mutex);
    g_unit_strips = unit_strips;
    return SDTW_OK;
}

int sdtw_set_reverse_mode(int dense) {
    std::lock_guard<std::mutex> lock(g_mutex);
    g_dense_reverse = dense ? 1 : 0;
    return SDTW_OK;
}

int sdtw_set_forward_rings(int on) {
    std::lock_guard<std::mutex> lock(g_mutex);
    if (on < 0 || on > 2) return SDTW_ERR_INVALID_ARG;
    g_forward_rings = on;
    return SDTW_OK;
}

int sdtw_set_reverse_kernel(int which) {
    if (which < -1 || which > 1) return SDTW_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_mutex);
    g_reverse_kernel = which;
    return SDTW_OK;
}

int sdtw_reverse_stats(uint64_t* chunks, uint64_t* skipped) {
    std::lock_guard<std::mutex> lock(g_mutex);
    unsigned long long h[2] = {0, 0};
    if (g_last_stats && g_last_stats_gen == g_ws_gen) {
        CUDA_TRY(cudaDeviceSynchronize());
        CUDA_TRY(cudaMemcpy(h, g_last_stats, sizeof(h), cudaMemcpyDeviceToHost));
    }
    if (chunks) *chunks = h[0];
    if (skipped) *skipped = h[1];
    return SDTW_OK;
}

int sdtw_tile_info(int32_t* cols_per_thread, int32_t* strip_cols, int32_t* ckpt_steps, int32_t* chunk_steps,
                   int32_t* rows_per_step) {
    if (rows_per_step) *rows_per_step = RP;
    if (cols_per_thread) *cols_per_thread = W;
    if (strip_cols) *strip_cols = SW;
    if (ckpt_steps) *ckpt_steps = TR;
    if (chunk_steps) *chunk_steps = CH;
    return SDTW_OK;
}

}  // extern "C"
