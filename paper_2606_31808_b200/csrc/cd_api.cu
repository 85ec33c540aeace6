// cd_api.cu -- the C ABI of include/cd.h: validation, automaton store, scratch management and
// kernel launches.  No torch types, no CPU fallback: every step of the path runs in the
// kernels of cd_step.cuh / cd_aux.cuh / cd_head.cuh / cd_dedup.cuh.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <string>
#include <utility>
#include <vector>

#include "../../include/cd.h"
#include "../../include/cd_diag.h"
#include "cd_aux.cuh"
#include "cd_common.cuh"
#include "cd_step.cuh"
#include "cd_head.cuh"
#include "cd_dedup.cuh"
#include "cd_types.hpp"

// NVTX ranges around every loop and every decoding step's enqueue: compiled in
// with -DCD_NVTX (python -m paper_2606_31808_b200.build --nvtx); header-only, nothing to link.
#ifdef CD_NVTX
#include <nvtx3/nvToolsExt.h>
#define CD_RANGE_PUSH(name) nvtxRangePushA(name)
#define CD_RANGE_POP() nvtxRangePop()
#else
#define CD_RANGE_PUSH(name) ((void)0)
#define CD_RANGE_POP() ((void)0)
#endif

namespace {

thread_local std::string g_err;
std::atomic<long long> g_launches{0};

cd_status fail(cd_status st, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return st;
}

#define CU(call)                                                                             \
    do {                                                                                     \
        cudaError_t e__ = (call);                                                            \
        if (e__ != cudaSuccess) {                                                            \
            const cd_status st__ = (e__ == cudaErrorMemoryAllocation) ? CD_ERR_OOM : CD_ERR_CUDA; \
            return fail(st__, "%s -> %s (%s:%d)", #call, cudaGetErrorString(e__), __FILE__, __LINE__); \
        }                                                                                    \
    } while (0)

struct RangeGuard {  // NVTX range for the scope (a no-op unless built with -DCD_NVTX)
    explicit RangeGuard(const char* name) { CD_RANGE_PUSH(name); (void)name; }
    ~RangeGuard() { CD_RANGE_POP(); }
};

// Launch shape of the step / loop kernels: 12 warps per CTA (one CTA per SM), 2 ring stages per warp,
// 8 KiB tiles = 192 KiB of logits in flight per SM.  Best or within noise of best on configs c1-c4 among
// the shapes swept in round 1 (profiles/r1_variant_sweep.md).
constexpr int STEP_WARPS = 12, STEP_STAGES = 2, STEP_TILE = 8192;
using StepRing = cd::WarpRing<STEP_STAGES, STEP_TILE>;

// Tuning knobs exist only in builds made with -DCD_TUNING (python -m paper_2606_31808_b200.build --tuning);
// the product reads no environment variable.
#ifdef CD_TUNING
int tune_int(const char* name, int def, int lo, int hi) {
    const char* e = std::getenv(name);
    if (!e) return def;
    const int v = std::atoi(e);
    return (v >= lo && v <= hi) ? v : def;
}
int tune_int_now(const char* name, int def) {
    const char* e = std::getenv(name);
    return e ? std::atoi(e) : def;
}
#else
constexpr int tune_int(const char*, int def, int, int) { return def; }
#endif

int units_per_warp() { static const int v = tune_int("CD_UPW", cd::UNITS_PER_WARP, 1, 32); return v; }
int tpu_max_tiles() { static const int v = tune_int("CD_TPU_MAX", cd::TPU_MAX_BYTES / STEP_TILE, 1, cd::TPU_MAX_BYTES / STEP_TILE); return v; }
bool use_pdl() { static const int v = tune_int("CD_PDL", 1, 0, 1); return v != 0; }
int flow_idle_ns() { static const int v = tune_int("CD_IDLE_NS", 32, 0, 100000); return v; }  // sleep between two polls of an unpublished task
bool head_pairs_enabled() { static const int v = tune_int("CD_HEAD_PAIRS", 1, 0, 1); return v != 0; }  // cta_group::2 kernel for > 128 dense rows
int host_gather_mult() { static const int v = tune_int("CD_HOST_GATHER_CTAS", 4, 1, 64); return v; }  // flat from 2 to 32 (51 GB/s on PCIe Gen5 x16)

// Per (handle, stream) scratch.  Operations on one stream are ordered, so one area per stream
// is race free; distinct streams get distinct areas.
struct StepBufs {  // sized by rows; replaced as a whole when the area grows
    int cap_rows = 0;
    long long cap_units = 0;
    cd::PartialSlot* partials = nullptr;
    int* tickets = nullptr;  // [rows] zero between launches
    int* ctrs = nullptr;  // [0] work, [1] finished CTAs, [2] errors of the running loop, [3] launch generation
    // per-step decode loops
    int* row_ids[2] = {nullptr, nullptr};
    int* state[2] = {nullptr, nullptr};
    int* state_new = nullptr;  // next states of a step launch
    int* n_active = nullptr;   // [2]
    int* token = nullptr;
    float* logprob = nullptr;
    uint8_t* done = nullptr;
    // persistent loop
    uint32_t* alive[3] = {nullptr, nullptr, nullptr};  // [ceil(rows / 32)] each
    int* state2[2] = {nullptr, nullptr};                // [rows] each
    int* bar = nullptr;                                 // [LB_INTS]
    unsigned long long* trace_t = nullptr;              // [LOOP_TRACE_STEPS + 1]
    int* trace_n = nullptr;                             // [LOOP_TRACE_STEPS + 1]
    unsigned long long* phase = nullptr;                // tuning builds: [LOOP_TRACE_STEPS][8]
    // flow_kernel (row tasks)
    int* f_q = nullptr;                                      // [FQ_INTS] see cd::FlowArgs
    unsigned long long* f_trace_t[2] = {nullptr, nullptr};  // [LOOP_TRACE_STEPS + 1] each
    int* f_trace_n[2] = {nullptr, nullptr};

    void release() {
        cudaFree(partials); cudaFree(tickets); cudaFree(ctrs);
        for (int i = 0; i < 2; ++i) { cudaFree(row_ids[i]); cudaFree(state[i]); cudaFree(state2[i]); }
        for (int i = 0; i < 3; ++i) cudaFree(alive[i]);
        cudaFree(state_new); cudaFree(n_active); cudaFree(token); cudaFree(logprob); cudaFree(done);
        cudaFree(bar); cudaFree(trace_t); cudaFree(trace_n); cudaFree(phase);
        cudaFree(f_q);
        for (int i = 0; i < 2; ++i) { cudaFree(f_trace_t[i]); cudaFree(f_trace_n[i]); }
        *this = StepBufs();
    }
};

struct Scratch {
    StepBufs b;
    // persistent loop: per-step work counters and the device copy of the step pointers
    int loop_steps_cap = 0;
    int* loop_work = nullptr;
    const void** loop_ptrs = nullptr;
    int trace_src = 0;  // the last loop on this stream ran in: 0 step_kernel launches, 1 loop_kernel, 2 flow_kernel
    unsigned long long* f_task = nullptr;  // flow_kernel: the task queue, [f_task_cap][4]
    long long f_task_cap = 0;
    int* h_status = nullptr;  // flow_kernel: [4] pinned, device-mapped host ints ([0] errors of the last loop, [1] its generation)
    int* d_status = nullptr;  //   the same memory as the device sees it
    // host-buffer loops
    void* stage[2] = {nullptr, nullptr};
    size_t stage_bytes[2] = {0, 0};
    int* out_i32 = nullptr;  // device copies of the host outputs
    size_t out_bytes = 0;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_copied[2] = {nullptr, nullptr};
    cudaEvent_t ev_consumed[2] = {nullptr, nullptr};
    int* h_pinned = nullptr;  // [8] pinned host ints
    int* h_ids = nullptr;     // [h_ids_cap] pinned host copy of the active row ids (host-buffer loop)
    int h_ids_cap = 0;
    // LM-head step (cd_head.cuh)
    int head_rows = 0, head_H = 0;
    uint8_t* h_flags = nullptr;   // [2 * rows]
    int* h_lists = nullptr;       // [4 * rows] dense slot / dense state / gather slot / gather state
    int* h_ctr = nullptr;         // [4]
    uint16_t* h_A = nullptr;      // [rows_pad, ldA]
    long long h_ldA = 0;
    cd::HeadPartial* h_partials = nullptr;
    cd::HeadPartial* h_gpartials = nullptr;  // [rows][HG_MAX_PIECES]
    CUtensorMap h_tmA{};

    void release_head() {
        cudaFree(h_flags); cudaFree(h_lists); cudaFree(h_ctr); cudaFree(h_A); cudaFree(h_partials); cudaFree(h_gpartials);
        h_flags = nullptr; h_lists = nullptr; h_ctr = nullptr; h_A = nullptr; h_partials = nullptr; h_gpartials = nullptr;
        head_rows = 0;
        head_H = 0;
    }
    void release() {
        b.release();
        release_head();
        cudaFree(loop_work); cudaFree(loop_ptrs); cudaFree(f_task);
        if (h_status) cudaFreeHost(h_status);
        for (int i = 0; i < 2; ++i) cudaFree(stage[i]);
        cudaFree(out_i32);
        if (copy_stream) cudaStreamDestroy(copy_stream);
        for (int i = 0; i < 2; ++i) {
            if (ev_copied[i]) cudaEventDestroy(ev_copied[i]);
            if (ev_consumed[i]) cudaEventDestroy(ev_consumed[i]);
        }
        if (h_pinned) cudaFreeHost(h_pinned);
        if (h_ids) cudaFreeHost(h_ids);
        *this = Scratch();
    }
};

// What the cd_set_* calls configure.  Every entry point takes a copy under the handle's mutex when it
// starts and works from that copy, so a setter never races with a call in progress: it applies to the
// calls that start after it returns.
struct Settings {
    int gather_max = 0;        // cd_set_gather_max: 0 dense scan only, > 0 threshold, < 0 automatic
    int head_gather_max = -1;  // cd_set_head_gather_max: 0 never gather, > 0 threshold, < 0 automatic
    float inv_tau = 0.0f;      // cd_set_sampling: 0 = greedy, else 1 / temperature
    unsigned long long seed = 0;
    int rng_step_base = 0;
    int limit = 0;             // cd_set_limit: LIMIT early exit applied by every loop entry point
    int* limit_ctr = nullptr;  //   device counter of satisfied rows (caller-owned); nullptr = no limit
    bool has_satisfying = false;  // cd_set_satisfying was called with a set
    int loop_mode = CD_LOOP_AUTO;  // cd_set_loop_mode: AUTO / PER_STEP / BARRIER
};

}  // namespace

struct cd_dfa {
    cd::DfaDev dev{};
    int device = 0;
    int start = 0;
    int start_accepting = 0;
    long long nnz = 0;
    int num_sms = 0;
    int coop_launch = 0;    // the device supports cooperative launches
    long long max_deg = 0;  // largest number of transitions of a state
    long long min_deg_nonacc = 0;  // fewest transitions of a non-accepting state
    void* d_mask = nullptr;
    void* d_row_ptr = nullptr;
    void* d_tok = nullptr;
    void* d_next = nullptr;
    void* d_acc = nullptr;
    void* d_rank = nullptr;
    void* d_satisfying = nullptr;  // [S], allocated with the handle, never freed before cd_free_dfa
    const void* w_ptr = nullptr;   // cached tensor map of the output embedding (cd_head_step)
    long long w_ld = 0;
    int w_H = 0;
    CUtensorMap w_tmap{};
    CUtensorMap w_tmap_half{};  // the same with boxes of HD_BN / 2 rows (CTA-pair kernel: each CTA loads half a W tile)
    std::mutex mu;  // guards cfg, the weight map cache and the scratch map
    Settings cfg;
    std::map<cudaStream_t, Scratch> scratch;
};

namespace {

Settings settings_of(const cd_dfa* d) {
    cd_dfa* dm = const_cast<cd_dfa*>(d);
    std::lock_guard<std::mutex> lk(dm->mu);
    return dm->cfg;
}

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceGuard() {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

int tiles_per_row(int V, int dtype) {
    const int tt = STEP_TILE / (dtype == CD_BF16 ? 2 : 4);
    return (V + tt - 1) / tt;
}

// Largest number of transitions a state may have to be gathered instead of scanned (0 = never).
// Automatic policy from the measured rates (profiles/r1d_gather_c4.md): the gather is transaction bound
// at ~31 G allowed logits/s (one scattered 2-byte logit per 64-byte DRAM granule), the dense scan streams
// a row at ~6.8 TB/s, so gathering pays while nnz / 31e9 < row_bytes / 6.8e12, i.e. nnz < row_bytes / 220;
// 232 leaves a margin so that states near the break-even stay on the dense path.
int gather_max_for(const cd_dfa* d, const Settings& cfg, int dtype) {
    if (cfg.gather_max >= 0) return cfg.gather_max;
    const long long row_bytes = (long long)d->dev.V * (dtype == CD_BF16 ? 2 : 4) + d->dev.V / 8;
    const long long g = row_bytes / 232;
    return (int)(g > 0x3FFFFFFF ? 0x3FFFFFFF : g);
}

int step_grid(const cd_dfa* d, long long n_upper, int dtype) {
    const long long tiles = n_upper * tiles_per_row(d->dev.V, dtype);
    long long g = (tiles + 1) / 2;  // few rows: still spread the tiles over many SMs
    if (g < 1) g = 1;
    if (g > d->num_sms) g = d->num_sms;
    return (int)g;
}

// chunk results of the step kernels: MAX_CHUNKS slots per row (cd_step.cuh: canonical chunks)
// = the most chunks (fp32 rows have the most tiles) or gathered pieces (any state may be gathered: cd_set_gather_max)
// a row of this automaton can have; a function of the automaton alone, so every launch on the handle agrees on it
int partial_stride(const cd_dfa* d) {
    const int chunks = cd::row_chunks(tiles_per_row(d->dev.V, CD_F32));
    // (gather_pieces is not monotone beyond MAX_CHUNKS * GATHER_CHUNK transitions: bound it)
    const long long p256 = (d->max_deg + cd::GATHER_CHUNK - 1) / cd::GATHER_CHUNK;
    const int pieces = (int)std::max<long long>(1, std::min<long long>(p256, cd::MAX_CHUNKS));
    return std::max(chunks, pieces);
}
long long step_units_cap(const cd_dfa* d, long long n) { return n * partial_stride(d) + 64; }

template <typename T>
cudaError_t dev_alloc(T** p, size_t count) {
    return cudaMalloc(reinterpret_cast<void**>(p), sizeof(T) * (count ? count : 1));
}

// Allocates a complete set of step buffers for `rows` rows; on failure nothing is kept.
cd_status alloc_step_bufs(const cd_dfa* d, int rows, StepBufs* out) {
    StepBufs n;
    const long long units = step_units_cap(d, rows);
    const size_t nwords = ((size_t)rows + 31) / 32;
    cudaError_t e = cudaSuccess;
    auto A = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
    A(dev_alloc(&n.partials, (size_t)units));
    A(dev_alloc(&n.ctrs, 4));
    A(dev_alloc(&n.tickets, 2 * (size_t)rows));
    for (int i = 0; i < 2; ++i) {
        A(dev_alloc(&n.row_ids[i], (size_t)rows));
        A(dev_alloc(&n.state[i], (size_t)rows));
        A(dev_alloc(&n.state2[i], (size_t)rows));
    }
    for (int i = 0; i < 3; ++i) A(dev_alloc(&n.alive[i], nwords));
    A(dev_alloc(&n.state_new, (size_t)rows));
    A(dev_alloc(&n.n_active, 2));
    A(dev_alloc(&n.token, (size_t)rows));
    A(dev_alloc(&n.logprob, (size_t)rows));
    A(dev_alloc(&n.done, (size_t)rows));
    A(dev_alloc(&n.bar, cd::LB_INTS));
    A(dev_alloc(&n.trace_t, (size_t)cd::LOOP_TRACE_STEPS + 1));
    A(dev_alloc(&n.trace_n, (size_t)cd::LOOP_TRACE_STEPS + 1));
    A(dev_alloc(&n.f_q, cd::FQ_INTS));
    for (int i = 0; i < 2; ++i) {
        A(dev_alloc(&n.f_trace_t[i], (size_t)cd::LOOP_TRACE_STEPS + 1));
        A(dev_alloc(&n.f_trace_n[i], (size_t)cd::LOOP_TRACE_STEPS + 1));
        if (e == cudaSuccess) e = cudaMemset(n.f_trace_t[i], 0, sizeof(unsigned long long) * ((size_t)cd::LOOP_TRACE_STEPS + 1));
        if (e == cudaSuccess) e = cudaMemset(n.f_trace_n[i], 0, sizeof(int) * ((size_t)cd::LOOP_TRACE_STEPS + 1));
    }
    if (e == cudaSuccess) e = cudaMemset(n.f_q, 0, sizeof(int) * cd::FQ_INTS);  // (the stop word 0 is never a launch generation)
#ifdef CD_TUNING
    A(dev_alloc(&n.phase, (size_t)cd::LOOP_TRACE_STEPS * 8));
#endif
    if (e == cudaSuccess) e = cudaMemset(n.partials, 0, sizeof(cd::PartialSlot) * (size_t)units);  // generation tags start at 0 ...
    if (e == cudaSuccess) {
        const int init[4] = {0, 0, 0, 1};  // ... launches at 1
        e = cudaMemcpy(n.ctrs, init, sizeof init, cudaMemcpyHostToDevice);
    }
    if (e == cudaSuccess) e = cudaMemset(n.tickets, 0, sizeof(int) * 2 * (size_t)rows);
    if (e == cudaSuccess) e = cudaMemset(n.trace_n, 0, sizeof(int) * ((size_t)cd::LOOP_TRACE_STEPS + 1));
    if (e != cudaSuccess) {
        n.release();
        return fail(e == cudaErrorMemoryAllocation ? CD_ERR_OOM : CD_ERR_CUDA, "scratch for %d rows: %s", rows,
                    cudaGetErrorString(e));
    }
    n.cap_units = units;
    n.cap_rows = rows;
    *out = n;
    return CD_OK;
}

cd_status get_scratch(const cd_dfa* cd_, cudaStream_t stream, int rows, Scratch** out) {
    cd_dfa* d = const_cast<cd_dfa*>(cd_);
    std::lock_guard<std::mutex> lk(d->mu);
    if ((long long)rows * (tiles_per_row(d->dev.V, CD_F32) + 1) >= 0x7FFFFFFFLL)
        return fail(CD_ERR_ARG, "rows (%d) * tiles per row overflows the unit index", rows);
    Scratch& s = d->scratch[stream];
    if (rows < 1) rows = 1;
    if (s.b.cap_rows < rows) {
        // growing: the new set is complete before the old one is touched; then wait for the work that
        // still uses the old buffers and drop them
        StepBufs fresh;
        const cd_status st = alloc_step_bufs(d, rows, &fresh);
        if (st != CD_OK) return st;
        if (s.b.cap_rows > 0) {
            const cudaError_t e = cudaStreamSynchronize(stream);
            if (e != cudaSuccess) {
                fresh.release();
                return fail(CD_ERR_CUDA, "cudaStreamSynchronize: %s", cudaGetErrorString(e));
            }
        }
        s.b.release();
        s.b = fresh;
        s.trace_src = 0;
        // The fresh counters restart the launch generation at 1, and flow_kernel's queue ring is tagged with
        // generations: entries left by earlier loops would read as already published.  The stream is idle here
        // (synchronised above if anything ever ran on these buffers): drop the ring, get_flow_scratch makes a
        // zeroed one.
        cudaFree(s.f_task);
        s.f_task = nullptr;
        s.f_task_cap = 0;
    }
    *out = &s;
    return CD_OK;
}

// grows a device buffer of the scratch area (contents are not kept); on failure the old buffer stays
cd_status grow_buffer(void** buf, size_t* have, size_t want, cudaStream_t stream) {
    if (*have >= want) return CD_OK;
    void* fresh = nullptr;
    CU(cudaMalloc(&fresh, want));
    const cudaError_t e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) {
        cudaFree(fresh);
        return fail(CD_ERR_CUDA, "cudaStreamSynchronize: %s", cudaGetErrorString(e));
    }
    cudaFree(*buf);
    *buf = fresh;
    *have = want;
    return CD_OK;
}

// staging + device copies of the outputs + copy stream / events of the host-buffer loops
cd_status get_host_loop_scratch(Scratch* s, size_t stage0_bytes, size_t stage1_bytes, size_t out_bytes, cudaStream_t stream) {
    cd_status st = grow_buffer(&s->stage[0], &s->stage_bytes[0], stage0_bytes, stream);
    if (st == CD_OK && stage1_bytes) st = grow_buffer(&s->stage[1], &s->stage_bytes[1], stage1_bytes, stream);
    if (st == CD_OK) st = grow_buffer(reinterpret_cast<void**>(&s->out_i32), &s->out_bytes, out_bytes, stream);
    if (st != CD_OK) return st;
    if (!s->copy_stream) CU(cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
        if (!s->ev_copied[i]) CU(cudaEventCreateWithFlags(&s->ev_copied[i], cudaEventDisableTiming));
        if (!s->ev_consumed[i]) CU(cudaEventCreateWithFlags(&s->ev_consumed[i], cudaEventDisableTiming));
    }
    if (!s->h_pinned) CU(cudaMallocHost(&s->h_pinned, sizeof(int) * 8));
    return CD_OK;
}

cd_status check_dtype(cd_dtype dt) {
    if (dt != CD_F32 && dt != CD_BF16) return fail(CD_ERR_ARG, "dtype must be CD_F32 or CD_BF16");
    return CD_OK;
}

template <int DT, bool GATHER = false, bool SAMPLE = false>
cd_status launch_step_t(const cd::StepArgs& a, int grid, cudaStream_t stream) {
    auto kern = cd::step_kernel<DT, STEP_WARPS, STEP_STAGES, STEP_TILE, GATHER, SAMPLE>;
    const size_t smem = sizeof(StepRing) * STEP_WARPS;
    static thread_local int configured_dev = -1;
    int dev = 0;
    CU(cudaGetDevice(&dev));
    if (configured_dev != dev) {
        CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        configured_dev = dev;
    }
    // programmatic stream serialization: this grid may be scheduled while the previous kernel
    // of the stream drains (the kernel itself waits with griddepcontrol.wait before touching
    // global memory), which hides the launch latency between the steps of a per-step decode loop
    cudaLaunchConfig_t lc{};
    lc.gridDim = dim3((unsigned)grid);
    lc.blockDim = dim3((unsigned)(STEP_WARPS * 32));
    lc.dynamicSmemBytes = smem;
    lc.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = use_pdl() ? 1 : 0;
    lc.attrs = at;
    lc.numAttrs = 1;
    CU(cudaLaunchKernelEx(&lc, kern, a));
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return CD_OK;
}

template <int DT>
cd_status launch_step_v(const cd::StepArgs& a, int grid, cudaStream_t stream) {
    if (a.inv_tau > 0.0f)  // sampling
        return a.gather_max > 0 ? launch_step_t<DT, true, true>(a, grid, stream)
                                : launch_step_t<DT, false, true>(a, grid, stream);
    if (a.gather_max > 0) return launch_step_t<DT, true>(a, grid, stream);  // density-adaptive rows
    return launch_step_t<DT>(a, grid, stream);
}

// Persistent loop: one cooperative launch (every CTA resident; they meet at a grid barrier after each
// decoding step).  *fits = false if the device cannot hold the grid (then the caller uses per-step launches).
template <int DT, bool GATHER = false, bool SAMPLE = false>
cd_status launch_loop_t(const cd::StepArgs& a, const cd::LoopArgs& L, int grid, cudaStream_t stream, bool* fits) {
    auto kern = cd::loop_kernel<DT, STEP_WARPS, STEP_STAGES, STEP_TILE, GATHER, SAMPLE>;
    const size_t nwords = ((size_t)L.B + 31) / 32;
    const size_t smem = sizeof(StepRing) * STEP_WARPS + ((2 * nwords + 1) * 4 + 15) / 16 * 16;
    static thread_local int configured_dev = -1;
    static thread_local int max_smem = 0;
    int dev = 0;
    CU(cudaGetDevice(&dev));
    if (configured_dev != dev) {
        CU(cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
        const size_t top = sizeof(StepRing) * STEP_WARPS + ((2 * ((size_t)cd::LOOP_MAX_ROWS / 32) + 1) * 4 + 15) / 16 * 16;
        CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(top < (size_t)max_smem ? top : (size_t)max_smem)));
        configured_dev = dev;
    }
    int per_sm = 0;
    if (smem <= (size_t)max_smem) CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, STEP_WARPS * 32, smem));
    int sms = 0;
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    *fits = per_sm >= 1 && (long long)per_sm * sms >= grid;
    if (!*fits) return CD_OK;
    cudaLaunchConfig_t lc{};
    lc.gridDim = dim3((unsigned)grid);
    lc.blockDim = dim3((unsigned)(STEP_WARPS * 32));
    lc.dynamicSmemBytes = smem;
    lc.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeCooperative;
    at[0].val.cooperative = 1;
    lc.attrs = at;
    lc.numAttrs = 1;
    CU(cudaLaunchKernelEx(&lc, kern, a, L));
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return CD_OK;
}

template <int DT>
cd_status launch_loop_v(const cd::StepArgs& a, const cd::LoopArgs& L, int grid, cudaStream_t stream, bool* fits) {
    if (a.inv_tau > 0.0f)
        return a.gather_max > 0 ? launch_loop_t<DT, true, true>(a, L, grid, stream, fits)
                                : launch_loop_t<DT, false, true>(a, L, grid, stream, fits);
    if (a.gather_max > 0) return launch_loop_t<DT, true>(a, L, grid, stream, fits);
    return launch_loop_t<DT>(a, L, grid, stream, fits);
}

// Persistent loop without a barrier (flow_kernel): a plain launch.  Its CTAs need not be resident together, but each
// of them must get to run (a warp's first unit is its global id): see FlowOrder for what that asks of the host.
template <int DT, bool GATHER = false, bool SAMPLE = false>
cd_status launch_flow_t(const cd::StepArgs& a, const cd::FlowArgs& F, int grid, cudaStream_t stream) {
    auto kern = cd::flow_kernel<DT, STEP_WARPS, STEP_STAGES, STEP_TILE, GATHER, SAMPLE>;
    const size_t smem = sizeof(StepRing) * STEP_WARPS;
    static thread_local int configured_dev = -1;
    int dev = 0;
    CU(cudaGetDevice(&dev));
    if (configured_dev != dev) {
        CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        configured_dev = dev;
    }
    // programmatic stream serialization (as launch_step_t): back-to-back loops of small batches (cd_decode_loop_async)
    // do not pay the launch latency between two kernels; the kernel waits (griddepcontrol.wait) before it touches
    // global memory, so whatever produced the logits has completed and flushed
    cudaLaunchConfig_t lc{};
    lc.gridDim = dim3((unsigned)grid);
    lc.blockDim = dim3((unsigned)(STEP_WARPS * 32));
    lc.dynamicSmemBytes = smem;
    lc.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = use_pdl() ? 1 : 0;
    lc.attrs = at;
    lc.numAttrs = 1;
    CU(cudaLaunchKernelEx(&lc, kern, a, F));
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return CD_OK;
}

template <int DT>
cd_status launch_flow_v(const cd::StepArgs& a, const cd::FlowArgs& F, int grid, cudaStream_t stream) {
    if (a.inv_tau > 0.0f)
        return a.gather_max > 0 ? launch_flow_t<DT, true, true>(a, F, grid, stream)
                                : launch_flow_t<DT, false, true>(a, F, grid, stream);
    if (a.gather_max > 0) return launch_flow_t<DT, true>(a, F, grid, stream);
    return launch_flow_t<DT>(a, F, grid, stream);
}

// Decode-loop extras of a step launch: per-row history + fused compaction (cd_step.cuh).
struct LoopExtras {
    int* tokens = nullptr;
    int* len = nullptr;
    int* final_state = nullptr;
    float* sum_logprob = nullptr;
    uint8_t* done = nullptr;
    int step = 0, max_steps = 0;
    int* row_ids_out = nullptr;
    int* state_out = nullptr;
    int* n_out = nullptr;
    const uint8_t* satisfying = nullptr;
    int* sat_ctr = nullptr;
    int limit = 0;
    int logits_by_slot = 0;
};

// the arguments every step launch shares (one cd_step, one step of a per-step loop, or the persistent loop)
cd::StepArgs make_step_args(const cd_dfa* d, const Settings& cfg, Scratch* s, cd_dtype dtype, long long ld,
                            const LoopExtras* x) {
    cd::StepArgs a{};
    if (x) {
        a.hist_tokens = x->tokens;
        a.hist_len = x->len;
        a.hist_final_state = x->final_state;
        a.hist_sum_logprob = x->sum_logprob;
        a.hist_done = x->done;
        a.step = x->step;
        a.max_steps = x->max_steps;
        a.cmp_row_ids_out = x->row_ids_out;
        a.cmp_state_out = x->state_out;
        a.cmp_n_out = x->n_out;
        a.satisfying = x->satisfying;
        a.sat_ctr = x->sat_ctr;
        a.limit = x->limit;
        a.logits_by_slot = x->logits_by_slot;
    }
    a.dfa = d->dev;
    a.ld_bytes = ld * (dtype == CD_BF16 ? 2 : 4);
    a.state_new = s->b.state_new;
    a.partials = s->b.partials;
    a.pstride = partial_stride(d);
    a.tickets = s->b.tickets;
    a.ctrs = s->b.ctrs;
    a.gather_max = gather_max_for(d, cfg, dtype);
    a.all_gather = (d->max_deg <= a.gather_max) ? 1 : 0;
    a.upw = units_per_warp();
    a.tpu_max = tpu_max_tiles();
    a.idle_ns = flow_idle_ns();
#ifdef CD_TUNING
    a.force_p = tune_int_now("CD_FORCE_P", 0);
#endif
    a.inv_tau = cfg.inv_tau;
    a.seed_lo = (uint32_t)(cfg.seed & 0xFFFFFFFFull);
    a.seed_hi = (uint32_t)(cfg.seed >> 32);
    a.rng_step_base = cfg.rng_step_base;
    return a;
}

// n_upper bounds the active count; n_dev (device int) overrides n inside the kernel.
cd_status launch_step(const cd_dfa* d, const Settings& cfg, Scratch* s, const void* logits, cd_dtype dtype, long long ld,
                      const int* row_map, int* state, int n_upper, const int* n_dev, int* token_out,
                      float* logprob_out, float* lse_out, uint8_t* done_out, cudaStream_t stream,
                      const LoopExtras* x = nullptr) {
    cd::StepArgs a = make_step_args(d, cfg, s, dtype, ld, x);
    a.logits = static_cast<const unsigned char*>(logits);
    a.row_map = row_map;
    a.state = state;
    a.n = n_upper;
    a.n_dev = n_dev;
    a.token_out = token_out;
    a.logprob_out = logprob_out;
    a.lse_out = lse_out;
    a.done_out = done_out;
    const int grid = step_grid(d, n_upper, dtype);
    return dtype == CD_BF16 ? launch_step_v<cd::DT_BF16>(a, grid, stream)
                            : launch_step_v<cd::DT_F32>(a, grid, stream);
}

cd_status check_logits_layout(const cd_dfa* d, const void* logits, cd_dtype dtype, long long ld) {
    const long long sz = dtype == CD_BF16 ? 2 : 4;
    if (!logits) return fail(CD_ERR_ARG, "logits is NULL");
    if (ld < d->dev.V) return fail(CD_ERR_ARG, "ld_elems (%lld) < V (%d)", ld, d->dev.V);
    if ((reinterpret_cast<uintptr_t>(logits) & 15) != 0) return fail(CD_ERR_ARG, "logits base is not 16-byte aligned");
    if ((ld * sz) % 16 != 0) return fail(CD_ERR_ARG, "row stride ld_elems*%lld is not a multiple of 16 bytes", sz);
    return CD_OK;
}

cd_status compile_impl(int32_t V, int32_t S, int32_t start, const int64_t* row_ptr, const int32_t* tok,
                       const int32_t* next, const uint8_t* accepting, int device, cd_dfa_t** out) {
    if (!out) return fail(CD_ERR_ARG, "out is NULL");
    if (V < 1 || S < 1) return fail(CD_ERR_ARG, "V and S must be >= 1 (V=%d S=%d)", V, S);
    if (!row_ptr || !accepting) return fail(CD_ERR_ARG, "row_ptr / accepting is NULL");
    // ---- validation
    if (start < 0 || start >= S) return fail(CD_ERR_AUTOMATON, "start state %d outside [0,%d)", start, S);
    if (row_ptr[0] != 0) return fail(CD_ERR_AUTOMATON, "row_ptr[0] = %lld, expected 0", (long long)row_ptr[0]);
    for (int32_t s = 0; s < S; ++s)
        if (row_ptr[s + 1] < row_ptr[s]) return fail(CD_ERR_AUTOMATON, "row_ptr decreases at state %d", s);
    const long long nnz = row_ptr[S];
    if (nnz > 0 && (!tok || !next)) return fail(CD_ERR_ARG, "tok / next is NULL with nnz = %lld", nnz);
    for (int32_t s = 0; s < S; ++s) {
        for (long long j = row_ptr[s]; j < row_ptr[s + 1]; ++j) {
            if (tok[j] < 0 || tok[j] >= V) return fail(CD_ERR_AUTOMATON, "state %d: token %d outside [0,%d)", s, tok[j], V);
            if (next[j] < 0 || next[j] >= S) return fail(CD_ERR_AUTOMATON, "state %d: next state %d outside [0,%d)", s, next[j], S);
            if (j > row_ptr[s] && tok[j] <= tok[j - 1]) return fail(CD_ERR_AUTOMATON, "state %d: tokens not strictly increasing", s);
        }
    }
    for (int32_t s = 0; s < S; ++s)
        if (row_ptr[s + 1] == row_ptr[s] && !accepting[s])
            return fail(CD_ERR_DEAD_STATE, "state %d is not accepting and has no transition", s);

    int ndev = 0;
    CU(cudaGetDeviceCount(&ndev));
    if (device < 0 || device >= ndev) return fail(CD_ERR_ARG, "device %d outside [0,%d)", device, ndev);
    DeviceGuard guard(device);
    if (!guard.ok) return fail(CD_ERR_CUDA, "cannot select device %d", device);

    cd_dfa* d = new (std::nothrow) cd_dfa();
    if (!d) return fail(CD_ERR_OOM, "host allocation failed");
    d->device = device;
    d->start = start;
    d->start_accepting = accepting[start] ? 1 : 0;
    d->nnz = nnz;
    d->min_deg_nonacc = nnz + 1;
    for (int32_t s = 0; s < S; ++s) {
        const long long deg = row_ptr[s + 1] - row_ptr[s];
        if (deg > d->max_deg) d->max_deg = deg;
        if (!accepting[s] && deg < d->min_deg_nonacc) d->min_deg_nonacc = deg;
    }
    cudaDeviceProp prop;
    cudaError_t e = cudaGetDeviceProperties(&prop, device);
    if (e != cudaSuccess) { delete d; return fail(CD_ERR_CUDA, "cudaGetDeviceProperties: %s", cudaGetErrorString(e)); }
    d->num_sms = prop.multiProcessorCount;
    d->coop_launch = prop.cooperativeLaunch;
    const int W = (V + 31) / 32;
    const int Wpad = (W + 3) & ~3;
    const int nblk = (V + 1023) / 1024;
    const size_t mask_bytes = (size_t)S * Wpad * 4;
    cd_status st = CD_OK;
    auto alloc = [&](void** p, size_t bytes) {
        if (st != CD_OK) return;
        cudaError_t e2 = cudaMalloc(p, bytes ? bytes : 16);
        if (e2 != cudaSuccess)
            st = fail(e2 == cudaErrorMemoryAllocation ? CD_ERR_OOM : CD_ERR_CUDA, "cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e2));
    };
    alloc(&d->d_mask, mask_bytes);
    alloc(&d->d_row_ptr, sizeof(long long) * (size_t)(S + 1));
    alloc(&d->d_tok, sizeof(int) * (size_t)nnz);
    alloc(&d->d_next, sizeof(int) * (size_t)nnz);
    alloc(&d->d_acc, (size_t)S);
    alloc(&d->d_rank, sizeof(int) * (size_t)S * nblk);
    alloc(&d->d_satisfying, (size_t)S);
    auto copy = [&](void* dst, const void* src, size_t bytes) {
        if (st != CD_OK || bytes == 0) return;
        cudaError_t e2 = cudaMemcpy(dst, src, bytes, cudaMemcpyHostToDevice);
        if (e2 != cudaSuccess) st = fail(CD_ERR_CUDA, "cudaMemcpy H2D: %s", cudaGetErrorString(e2));
    };
    static_assert(sizeof(long long) == sizeof(int64_t), "row_ptr width");
    copy(d->d_row_ptr, row_ptr, sizeof(long long) * (size_t)(S + 1));
    copy(d->d_tok, tok, sizeof(int) * (size_t)nnz);
    copy(d->d_next, next, sizeof(int) * (size_t)nnz);
    copy(d->d_acc, accepting, (size_t)S);
    if (st == CD_OK) {
        cudaError_t e2 = cudaMemset(d->d_mask, 0, mask_bytes);
        if (e2 == cudaSuccess) e2 = cudaMemset(d->d_satisfying, 0, (size_t)S);
        const int threads = 256;
        long long blocks = ((long long)S * 32 + threads - 1) / threads;
        if (blocks > 65535) blocks = 65535;
        if (e2 == cudaSuccess && nnz > 0) {
            cd::build_mask_kernel<<<(int)blocks, threads>>>(static_cast<const long long*>(d->d_row_ptr),
                                                           static_cast<const int*>(d->d_tok),
                                                           static_cast<int*>(d->d_next),
                                                           static_cast<const uint8_t*>(d->d_acc), S, Wpad,
                                                           static_cast<uint32_t*>(d->d_mask));
            g_launches.fetch_add(1, std::memory_order_relaxed);
            e2 = cudaGetLastError();
        }
        if (e2 == cudaSuccess) {
            cd::build_rank_kernel<<<(int)blocks, threads>>>(static_cast<const uint32_t*>(d->d_mask), S, Wpad, nblk,
                                                           static_cast<int*>(d->d_rank));
            g_launches.fetch_add(1, std::memory_order_relaxed);
            e2 = cudaGetLastError();
        }
        if (e2 == cudaSuccess) e2 = cudaDeviceSynchronize();
        if (e2 != cudaSuccess) st = fail(CD_ERR_CUDA, "mask build: %s", cudaGetErrorString(e2));
    }
    if (st != CD_OK) {
        cudaFree(d->d_mask); cudaFree(d->d_row_ptr); cudaFree(d->d_tok); cudaFree(d->d_next); cudaFree(d->d_acc);
        cudaFree(d->d_rank); cudaFree(d->d_satisfying);
        delete d;
        return st;
    }
    d->dev.V = V;
    d->dev.S = S;
    d->dev.W = W;
    d->dev.Wpad = Wpad;
    d->dev.mask = static_cast<const uint32_t*>(d->d_mask);
    d->dev.row_ptr = static_cast<const long long*>(d->d_row_ptr);
    d->dev.tok = static_cast<const int*>(d->d_tok);
    d->dev.next = static_cast<const int*>(d->d_next);
    d->dev.accepting = static_cast<const uint8_t*>(d->d_acc);
    d->dev.rank1k = static_cast<const int*>(d->d_rank);
    d->dev.nblk = nblk;
    *out = d;
    return CD_OK;
}

cd_status compile_csr(int32_t V, const cdt::HostCsr& c, int device, cd_dfa_t** out) {
    return compile_impl(V, c.S, 0, c.row_ptr.data(), c.tok.data(), c.next.data(), c.accepting.data(), device, out);
}

cd_status copy_csr_out(const cdt::HostCsr& c, int32_t* S_out, int64_t* nnz_out, int64_t* row_ptr_out, int32_t* tok_out,
                       int32_t* next_out, uint8_t* accepting_out) {
    *S_out = c.S;
    *nnz_out = (int64_t)c.tok.size();
    if (row_ptr_out) std::memcpy(row_ptr_out, c.row_ptr.data(), sizeof(int64_t) * c.row_ptr.size());
    if (tok_out && !c.tok.empty()) std::memcpy(tok_out, c.tok.data(), sizeof(int32_t) * c.tok.size());
    if (next_out && !c.next.empty()) std::memcpy(next_out, c.next.data(), sizeof(int32_t) * c.next.size());
    if (accepting_out) std::memcpy(accepting_out, c.accepting.data(), c.accepting.size());
    return CD_OK;
}

struct LimitArgs {
    int* sat_ctr = nullptr;  // device counter; nullptr = no limit
    int limit = 0;
};

// the LIMIT a loop runs under: the explicit one (cd_decode_loop_limit), else the handle's (cd_set_limit)
LimitArgs resolve_limit(const Settings& cfg, const LimitArgs& explicit_lim = LimitArgs()) {
    if (explicit_lim.sat_ctr) return explicit_lim;
    LimitArgs l;
    if (cfg.limit_ctr && cfg.has_satisfying) {
        l.sat_ctr = cfg.limit_ctr;
        l.limit = cfg.limit;
    }
    return l;
}

// persist: also initialise the bitmaps / states / counters of loop_kernel
cd_status launch_loop_init(const cd_dfa* d, Scratch* s, int B, int max_steps, int* tokens_out, int* len_out,
                           int* final_state_out, float* sum_logprob_out, uint8_t* done_out, cudaStream_t stream,
                           const LimitArgs& lim = LimitArgs(), bool persist = false) {
    long long work = (long long)B * (max_steps > 0 ? max_steps : 1);
    long long blocks = (work + 255) / 256;
    if (blocks < 1) blocks = 1;
    if (blocks > 4096) blocks = 4096;
    cd::LoopInitArgs a{};
    a.B = B;
    a.max_steps = max_steps;
    a.start = d->start;
    a.start_accepting = d->start_accepting;
    a.tokens_out = tokens_out;
    a.len_out = len_out;
    a.final_state_out = final_state_out;
    a.sum_logprob_out = sum_logprob_out;
    a.done_row_out = done_out;
    a.sat_ctr = lim.sat_ctr;
    a.limit = lim.limit;
    a.ctrs = s->b.ctrs;
    if (persist) {
        for (int i = 0; i < 3; ++i) a.alive[i] = s->b.alive[i];
        for (int i = 0; i < 2; ++i) a.state2[i] = s->b.state2[i];
        a.work = s->loop_work;
        a.bar = s->b.bar;
    } else {
        a.row_ids = s->b.row_ids[0];
        a.state = s->b.state[0];
        a.n_active = s->b.n_active;
    }
    cd::loop_init_kernel<<<(int)blocks, 256, 0, stream>>>(a);
    CU(cudaGetLastError());
    g_launches.fetch_add(1, std::memory_order_relaxed);
    s->trace_src = 0;
    return CD_OK;
}

// One iteration k of a per-step loop on `logits` ([B, ld], original row ids): ONE launch -- the step
// kernel records the per-row history as rows finalise and its last CTA compacts the active list.
cd_status enqueue_loop_step(const cd_dfa* d, const Settings& cfg, Scratch* s, const void* logits, cd_dtype dtype,
                            long long ld, int B, int k, int max_steps, int* tokens_out, int* len_out,
                            int* final_state_out, float* sum_logprob_out, uint8_t* done_out, cudaStream_t stream,
                            const LimitArgs& lim = LimitArgs(), int logits_by_slot = 0) {
    RangeGuard range("cd decoding step");
    const int cur = k & 1, nxt = cur ^ 1;
    LoopExtras x;
    x.logits_by_slot = logits_by_slot;
    if (lim.sat_ctr) {
        x.satisfying = static_cast<const uint8_t*>(d->d_satisfying);
        x.sat_ctr = lim.sat_ctr;
        x.limit = lim.limit;
    }
    x.tokens = tokens_out;
    x.len = len_out;
    x.final_state = final_state_out;
    x.sum_logprob = sum_logprob_out;
    x.done = done_out;
    x.step = k;
    x.max_steps = max_steps;
    x.row_ids_out = s->b.row_ids[nxt];
    x.state_out = s->b.state[nxt];
    x.n_out = s->b.n_active + nxt;
    return launch_step(d, cfg, s, logits, dtype, ld, s->b.row_ids[cur], s->b.state[cur], B, s->b.n_active + cur,
                       s->b.token, s->b.logprob, nullptr, s->b.done, stream, &x);
}

// The whole loop in ONE cooperative launch (cd_step.cuh loop_kernel).  *launched = false when this loop
// cannot take that path (too many rows for the bitmap snapshot, no cooperative launch, CTAs do not fit):
// the caller then enqueues per-step launches.
cd_status enqueue_persistent_loop(const cd_dfa* d, const Settings& cfg, Scratch* s, const void* const* step_logits,
                                  cd_dtype dtype, long long ld, int B, int max_steps, int* tokens_out, int* len_out,
                                  int* final_state_out, float* sum_logprob_out, uint8_t* done_out, cudaStream_t stream,
                                  const LimitArgs& lim, bool* launched) {
    RangeGuard range("cd decode loop (persistent kernel)");
    *launched = false;
    LoopExtras x;
    if (lim.sat_ctr) {
        x.satisfying = static_cast<const uint8_t*>(d->d_satisfying);
        x.sat_ctr = lim.sat_ctr;
        x.limit = lim.limit;
    }
    x.tokens = tokens_out;
    x.len = len_out;
    x.final_state = final_state_out;
    x.sum_logprob = sum_logprob_out;
    x.done = done_out;
    x.max_steps = max_steps;
    cd::StepArgs a = make_step_args(d, cfg, s, dtype, ld, &x);
    a.n = B;
    cd::LoopArgs L{};
    if (max_steps <= cd::LOOP_PARAM_STEPS) {
        for (int k = 0; k < max_steps; ++k) L.step_ptrs[k] = step_logits[k];
    } else {
        CU(cudaMemcpyAsync(s->loop_ptrs, step_logits, sizeof(void*) * (size_t)max_steps, cudaMemcpyHostToDevice, stream));
        L.step_ptrs_dev = s->loop_ptrs;
    }
    L.B = B;
    for (int i = 0; i < 3; ++i) L.alive[i] = s->b.alive[i];
    for (int i = 0; i < 2; ++i) L.state2[i] = s->b.state2[i];
    L.work = s->loop_work;
    L.bar = s->b.bar;
    L.trace_t = s->b.trace_t;
    L.trace_n = s->b.trace_n;
#ifdef CD_TUNING
    L.phase = s->b.phase;
    CU(cudaMemsetAsync(s->b.phase, 0, sizeof(unsigned long long) * (size_t)cd::LOOP_TRACE_STEPS * 8, stream));
#endif
    const int grid = step_grid(d, B, dtype);
    const cd_status st = dtype == CD_BF16 ? launch_loop_v<cd::DT_BF16>(a, L, grid, stream, launched)
                                          : launch_loop_v<cd::DT_F32>(a, L, grid, stream, launched);
    if (st == CD_OK && *launched) s->trace_src = 1;
    return st;
}

cd_status get_loop_scratch(Scratch* s, int max_steps, cudaStream_t stream);

// Order of flow_kernel launches on one device across the streams of this process.  While the process has used a
// single stream for these loops nothing is added: stream order does it, and back-to-back loops keep their
// programmatic overlap.  When a second stream shows up the device is synchronised once; from then on every launch
// records an event and a launch on another stream waits for the one before it.  Loops of OTHER PROCESSES on the
// same GPU are not covered: they can starve each other into the idle timeout (CD_ERR_INTERNAL), see cd.h.
struct FlowOrder {
    std::mutex mu;
    cudaStream_t last = nullptr;
    bool any = false, multi = false, ev_recorded = false;
    cudaEvent_t ev = nullptr;
};
FlowOrder& flow_order(int dev) {
    static FlowOrder o[64];
    return o[dev & 63];
}

// flow_kernel: whether the loop fits the kernel's index ranges
constexpr long long FLOW_RING_MAX = (512ll << 20) / (8 * cd::FLOW_ENTRY_WORDS);  // at most 512 MiB of queue

// entries of the queue ring: a power of two >= 2 * B * (chunks per row): a row step is cut into at most that many units
// (see cd::FlowArgs: B * chunks suffices)
long long flow_ring_entries(const cd_dfa* d, int B, int dtype) {
    const long long tc = cd::row_chunks(tiles_per_row(d->dev.V, dtype));
    long long cap = 1024;
    while (cap < 2ll * B * tc) cap <<= 1;
    return cap;
}

bool flow_loop_possible(const cd_dfa* d, int B, int max_steps, int dtype) {
    if (flow_ring_entries(d, B, dtype) > FLOW_RING_MAX) return false;
    // the unit counter and the entry counter are 32 bits wide: every row step cut into MAX_CHUNKS units at worst
    return (long long)B * max_steps * cd::MAX_CHUNKS + (long long)d->num_sms * STEP_WARPS * 4 < 0x7FFFFFFFLL;
}

// status word of the loops (pinned, device-mapped host memory)
cd_status get_status_word(Scratch* s) {
    if (!s->h_status) {
        CU(cudaHostAlloc(reinterpret_cast<void**>(&s->h_status), sizeof(int) * 4, cudaHostAllocMapped | cudaHostAllocPortable));
        std::memset(s->h_status, 0, sizeof(int) * 4);
        if (cudaHostGetDevicePointer(reinterpret_cast<void**>(&s->d_status), s->h_status, 0) != cudaSuccess) {
            cudaFreeHost(s->h_status);
            s->h_status = nullptr;
            return fail(CD_ERR_CUDA, "mapped status word");
        }
    }
    return CD_OK;
}

// queue ring + status word of flow_kernel
cd_status get_flow_scratch(Scratch* s, long long entries, cudaStream_t stream) {
    const cd_status st = get_status_word(s);
    if (st != CD_OK) return st;
    if (s->f_task_cap >= entries) return CD_OK;
    unsigned long long* q = nullptr;
    if (dev_alloc(&q, (size_t)entries * cd::FLOW_ENTRY_WORDS) != cudaSuccess)
        return fail(CD_ERR_OOM, "queue of %lld entries", entries);
    if (cudaMemset(q, 0, sizeof(unsigned long long) * cd::FLOW_ENTRY_WORDS * (size_t)entries) != cudaSuccess) {  // tags start at 0
        cudaFree(q);
        return fail(CD_ERR_CUDA, "queue");
    }
    if (s->f_task) cudaStreamSynchronize(stream);
    cudaFree(s->f_task);
    s->f_task = q;
    s->f_task_cap = entries;
    return CD_OK;
}

// The whole loop in ONE launch of flow_kernel and nothing else: no set-up kernel, no copy afterwards (no LIMIT:
// a LIMIT is defined step by step over all rows, which needs the lock-step of loop_kernel).
cd_status enqueue_flow_loop(const cd_dfa* d, const Settings& cfg, Scratch* s, const void* const* step_logits,
                            cd_dtype dtype, long long ld, int B, int max_steps, int* tokens_out, int* len_out,
                            int* final_state_out, float* sum_logprob_out, uint8_t* done_out, cudaStream_t stream) {
    RangeGuard range("cd decode loop (persistent kernel, row tasks)");
    cd_status st = get_flow_scratch(s, flow_ring_entries(d, B, dtype), stream);
    if (st != CD_OK) return st;
    LoopExtras x;
    x.tokens = tokens_out;
    x.len = len_out;
    x.final_state = final_state_out;
    x.sum_logprob = sum_logprob_out;
    x.done = done_out;
    x.max_steps = max_steps;
    cd::StepArgs a = make_step_args(d, cfg, s, dtype, ld, &x);
    a.n = B;
    const int grid = step_grid(d, B, dtype);
    cd::FlowArgs F{};
    if (max_steps <= cd::LOOP_PARAM_STEPS) {
        for (int k = 0; k < max_steps; ++k) F.step_ptrs[k] = step_logits[k];
    } else {
        st = get_loop_scratch(s, max_steps, stream);
        if (st != CD_OK) return st;
        CU(cudaMemcpyAsync(s->loop_ptrs, step_logits, sizeof(void*) * (size_t)max_steps, cudaMemcpyHostToDevice, stream));
        F.step_ptrs_dev = s->loop_ptrs;
    }
    F.B = B;
    F.start = d->start;
    F.task = s->f_task;
    {  // the ring in use: the largest power of two the allocation holds (it only ever grows)
        int lg = 0;
        while ((2ll << lg) <= s->f_task_cap) ++lg;
        F.cap_log2 = lg;
        F.cap_mask = (unsigned)((1ll << lg) - 1);
    }
    {  // units a published row step is cut into (cd::FlowArgs): 64 / 32 / 16 KiB units or every chunk
        const int T = tiles_per_row(d->dev.V, dtype), ct = cd::chunk_tiles(T), tc = cd::row_chunks(T);
        const int W = grid * STEP_WARPS;
        int tiles[4] = {tpu_max_tiles(), tpu_max_tiles() / 2, tpu_max_tiles() / 4, 1};
        int th[3] = {0, -W / 2, -(W * 9) / 10};  // (c3: 530 us per loop against 538 with W/2, 0, -W/2; c2 / c4 the same)
#ifdef CD_TUNING
        if (const char* e = std::getenv("CD_FLOW_TILES")) std::sscanf(e, "%d,%d,%d,%d", &tiles[0], &tiles[1], &tiles[2], &tiles[3]);
        if (const char* e = std::getenv("CD_FLOW_TH")) {  // in percent of the warps
            int p[3] = {0, -50, -90};
            std::sscanf(e, "%d,%d,%d", &p[0], &p[1], &p[2]);
            for (int i = 0; i < 3; ++i) th[i] = (int)((long long)W * p[i] / 100);
        }
#endif
        for (int i = 0; i < 4; ++i) {
            const int cpu = std::max(1, tiles[i] / ct);
            F.np_lvl[i] = (tc + cpu - 1) / cpu;
        }
        for (int i = 0; i < 3; ++i) F.th[i] = th[i];
    }
    F.q = s->b.f_q;
    for (int i = 0; i < 2; ++i) {
        F.trace_t[i] = s->b.f_trace_t[i];
        F.trace_n[i] = s->b.f_trace_n[i];
    }
    F.host_status = s->d_status;
#ifdef CD_TUNING
    if (const char* e = std::getenv("CD_DBG_PTR")) {  // a device buffer of the caller's, [CD_DBG_CAP][8] u64, zeroed
        F.dbg = reinterpret_cast<unsigned long long*>(std::strtoull(e, nullptr, 0));
        F.dbg_cap = tune_int_now("CD_DBG_CAP", 0);
    }
#endif
    {
        // flow_kernel hands every warp its first unit by global warp id, so a launch ends only once ALL of its CTAs
        // have run.  Two launches on two streams could each hold part of the SMs and wait for the rest until the
        // idle timeout; launches on a device are therefore ordered across the streams of this process (FlowOrder).
        FlowOrder& fo = flow_order(d->device);
        std::lock_guard<std::mutex> lk(fo.mu);
        if (fo.any && fo.last != stream) {
            if (!fo.multi) {  // the second stream this process uses for these loops: from now on launches leave an event
                CU(cudaDeviceSynchronize());
                CU(cudaEventCreateWithFlags(&fo.ev, cudaEventDisableTiming));
                fo.multi = true;
            } else if (fo.ev_recorded) {
                CU(cudaStreamWaitEvent(stream, fo.ev, 0));
            }
        }
        st = dtype == CD_BF16 ? launch_flow_v<cd::DT_BF16>(a, F, grid, stream) : launch_flow_v<cd::DT_F32>(a, F, grid, stream);
        if (st == CD_OK) {
            if (fo.multi && cudaEventRecord(fo.ev, stream) == cudaSuccess) fo.ev_recorded = true;
            fo.last = stream;
            fo.any = true;
        }
    }
    if (st == CD_OK) s->trace_src = 2;
    return st;
}

// A loop that gave up (a row that never finished, a merge that timed out) leaves the tickets of its unfinished row
// steps non-zero; the next loop on this scratch would count from them and merge too early.  Back to zero, in
// stream order, before anything else runs on these buffers.
void clear_tickets(Scratch* s, cudaStream_t stream) {
    if (s->b.tickets) cudaMemsetAsync(s->b.tickets, 0, sizeof(int) * 2 * (size_t)s->b.cap_rows, stream);
}

// End of a flow_kernel loop: the one stream synchronisation the loops promise; the kernel has put its status
// into mapped host memory.
cd_status finish_flow_loop(Scratch* s, cudaStream_t stream) {
    CU(cudaStreamSynchronize(stream));
    if (!s->h_status) return CD_OK;
    const int err = reinterpret_cast<volatile int*>(s->h_status)[0];
    reinterpret_cast<volatile int*>(s->h_status)[0] = 0;
    if (err != 0) clear_tickets(s, stream);
    if (err != 0)
        return fail(CD_ERR_INTERNAL, "%d device-side consistency failures (state out of range, token missing from the CSR or a row that never finished)", err);
    return CD_OK;
}

std::mutex& coop_mutex(int dev) {
    static std::mutex mu[64];
    return mu[dev & 63];
}

// can this loop run in loop_kernel at all?  (the launch itself still checks that the CTAs fit)
bool persistent_loop_possible(const cd_dfa* d, const Settings& cfg, int B, int max_steps) {
    return cfg.loop_mode != CD_LOOP_PER_STEP && d->coop_launch && B <= cd::LOOP_MAX_ROWS && max_steps > 0 &&
           max_steps < (1 << 24) && !d->start_accepting;
}

// per-step work counters / device step pointers of the persistent loop
cd_status get_loop_scratch(Scratch* s, int max_steps, cudaStream_t stream) {
    if (s->loop_steps_cap >= max_steps) return CD_OK;
    int* work = nullptr;
    const void** ptrs = nullptr;
    const int cap = max_steps < 64 ? 64 : max_steps;
    CU(dev_alloc(&work, (size_t)cap));
    if (dev_alloc(&ptrs, (size_t)cap) != cudaSuccess) {
        cudaFree(work);
        return fail(CD_ERR_OOM, "loop scratch for %d steps", max_steps);
    }
    if (s->loop_steps_cap > 0) cudaStreamSynchronize(stream);
    cudaFree(s->loop_work);
    cudaFree(s->loop_ptrs);
    s->loop_work = work;
    s->loop_ptrs = ptrs;
    s->loop_steps_cap = cap;
    return CD_OK;
}

// Stream-ordered scratch (cudaMallocAsync) must not be handed back to the OS at every synchronisation:
// keep the default pool's memory (once per device).
void keep_pool_memory(int dev) {
    static std::mutex mu;
    static std::map<int, bool> done;
    std::lock_guard<std::mutex> lk(mu);
    if (done[dev]) return;
    cudaMemPool_t pool = nullptr;
    if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess && pool) {
        unsigned long long thr = ~0ull;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
    }
    done[dev] = true;
}

cd_status device_of(const void* p, int* dev) {
    cudaPointerAttributes at;
    CU(cudaPointerGetAttributes(&at, p));
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
        return fail(CD_ERR_ARG, "expected a DEVICE pointer");
    *dev = at.device;
    return CD_OK;
}

// Stable compaction of n slots (a6): one CTA up to one chunk (no allocation: capturable in a CUDA graph),
// above that the single-pass look-back kernel over ceil(n / 4096) CTAs with stream-ordered scratch for the
// chunk states.  rank_out: see compact_lookback_kernel.
cd_status launch_compact(const uint8_t* done, const int* row_ids_in, const int* state_in, int n, int* row_ids_out,
                         int* state_out, int* n_out, int* rank_out, cudaStream_t stream) {
    if (n <= cd::SCAN_CHUNK && !rank_out) {
        cd::compact_kernel<<<1, 1024, 0, stream>>>(done, row_ids_in, state_in, n, row_ids_out, state_out, n_out);
        CU(cudaGetLastError());
        g_launches.fetch_add(1, std::memory_order_relaxed);
        return CD_OK;
    }
    int dev = 0;
    cd_status st = device_of(n_out, &dev);
    if (st != CD_OK) return st;
    DeviceGuard guard(dev);
    keep_pool_memory(dev);
    const int chunks = n > 0 ? (n + cd::SCAN_CHUNK - 1) / cd::SCAN_CHUNK : 1;
    const size_t bytes = sizeof(unsigned long long) * ((size_t)chunks + 1);
    unsigned long long* tile = nullptr;
    CU(cudaMallocAsync(reinterpret_cast<void**>(&tile), bytes, stream));
    cudaError_t e = cudaMemsetAsync(tile, 0, bytes, stream);
    if (e == cudaSuccess) {
        cd::compact_lookback_kernel<<<chunks, 1024, 0, stream>>>(done, row_ids_in, state_in, n, row_ids_out, state_out,
                                                                n_out, rank_out, tile, reinterpret_cast<int*>(tile + chunks));
        e = cudaGetLastError();
    }
    cudaFreeAsync(tile, stream);  // on every path
    if (e != cudaSuccess) return fail(CD_ERR_CUDA, "compaction launch: %s", cudaGetErrorString(e));
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return CD_OK;
}

// ---- cd_compact_noalloc (include/cd.h): the look-back compaction with its chunk words in the library image.
// A caller that shares the GPU with an LM server holding nearly all of HBM, or that runs without a usable
// memory pool, cannot afford launch_compact's cudaMallocAsync; this array is the scratch it gets instead.
// One word per 4096-slot chunk + the ticket word behind the words in use: 4097 x 8 = 32,776 bytes on every
// GPU that loads the library, until the process exits.  Shared by all calls on a GPU (see the header).
constexpr int NOALLOC_MAX_CHUNKS = CD_COMPACT_NOALLOC_MAX_N / cd::SCAN_CHUNK;
static_assert(CD_COMPACT_NOALLOC_MAX_N % cd::SCAN_CHUNK == 0, "the limit is a whole number of chunks");
static __device__ __align__(256) unsigned long long g_noalloc_tiles[NOALLOC_MAX_CHUNKS + 1];

// In host code `g_noalloc_tiles` is only a handle for the runtime, not an address a kernel may use: the
// device address is asked for once per GPU, with that GPU current, and kept.  No allocation afterwards.
constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mu;
unsigned long long* g_noalloc_addr[NOALLOC_MAX_DEVICES] = {};

cd_status noalloc_tiles_of(int dev, unsigned long long** out) {  // `dev` is the current device
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(CD_ERR_ARG, "cd_compact_noalloc: device ordinal %d not supported", dev);
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    if (!g_noalloc_addr[dev]) {
        void* p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_noalloc_tiles));
        if (!p) return fail(CD_ERR_CUDA, "cd_compact_noalloc: no device address for the scratch array on device %d", dev);
        g_noalloc_addr[dev] = static_cast<unsigned long long*>(p);
    }
    *out = g_noalloc_addr[dev];
    return CD_OK;
}

cd_status launch_compact_noalloc(const uint8_t* done, const int* row_ids_in, const int* state_in, int n, int* row_ids_out,
                                 int* state_out, int* n_out, cudaStream_t stream) {
    int dev = 0;
    cd_status st = device_of(n_out, &dev);
    if (st != CD_OK) return st;
    DeviceGuard guard(dev);
    if (!guard.ok) return fail(CD_ERR_CUDA, "cd_compact_noalloc: cannot make device %d current", dev);
    unsigned long long* tile = nullptr;
    st = noalloc_tiles_of(dev, &tile);
    if (st != CD_OK) return st;
    const int chunks = n > 0 ? (n + cd::SCAN_CHUNK - 1) / cd::SCAN_CHUNK : 1;
    // the words of this call (chunk states + ticket) still hold the last call's prefixes: back to zero, in stream order
    CU(cudaMemsetAsync(tile, 0, sizeof(unsigned long long) * ((size_t)chunks + 1), stream));
    cd::compact_lookback_kernel<<<chunks, 1024, 0, stream>>>(done, row_ids_in, state_in, n, row_ids_out, state_out, n_out,
                                                            nullptr, tile, reinterpret_cast<int*>(tile + chunks));
    CU(cudaGetLastError());
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return CD_OK;
}

// End of every loop: one read of the error counter (and of the persistent loop's abort flag) and the one
// stream synchronisation the loops promise.
cd_status finish_loop(Scratch* s, cudaStream_t stream, bool persistent) {
    int h[4] = {0, 0, 0, 0};
    int hb[4] = {0, 0, 0, 0};
    CU(cudaMemcpyAsync(h, s->b.ctrs, sizeof h, cudaMemcpyDeviceToHost, stream));
    if (persistent) CU(cudaMemcpyAsync(hb + 2, s->b.bar + cd::LB_ABORT, sizeof(int), cudaMemcpyDeviceToHost, stream));
    CU(cudaStreamSynchronize(stream));
    if (hb[2] != 0 || h[2] != 0) clear_tickets(s, stream);
    if (hb[2] != 0)
        return fail(CD_ERR_INTERNAL, "the persistent loop kernel timed out at a grid barrier (device shared with a kernel that never ends?)");
    if (h[2] != 0)
        return fail(CD_ERR_INTERNAL, "%d device-side consistency failures (state out of range or token missing from the CSR)", h[2]);
    return CD_OK;
}

}  // namespace

// =============================================================================== C ABI
extern "C" {

const char* cd_last_error(void) { return g_err.c_str(); }

int64_t cd_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

cd_status cd_compile_dfa(int32_t V, int32_t S, int32_t start, const int64_t* row_ptr, const int32_t* tok,
                         const int32_t* next, const uint8_t* accepting, int device, cd_dfa_t** out) {
    try {
        return compile_impl(V, S, start, row_ptr, tok, next, accepting, device, out);
    } catch (const std::bad_alloc&) {
        return fail(CD_ERR_OOM, "host allocation failed");
    } catch (...) {
        return fail(CD_ERR_INTERNAL, "unexpected exception");
    }
}

cd_status cd_build_trie(int32_t V, int32_t K, const int64_t* label_ptr, const int32_t* label_tok, int32_t eos,
                        int32_t* S_out, int64_t* nnz_out, int64_t* row_ptr_out, int32_t* tok_out, int32_t* next_out,
                        uint8_t* accepting_out) {
    try {
        if (!label_ptr || !S_out || !nnz_out) return fail(CD_ERR_ARG, "NULL argument");
        if (V < 1 || K < 1) return fail(CD_ERR_ARG, "V and K must be >= 1");
        if (label_ptr[K] > 0 && !label_tok) return fail(CD_ERR_ARG, "label_tok is NULL");
        cdt::HostCsr c;
        const std::string err = cdt::build_trie(V, K, label_ptr, label_tok, eos, &c);
        if (!err.empty()) return fail(CD_ERR_AUTOMATON, "%s", err.c_str());
        return copy_csr_out(c, S_out, nnz_out, row_ptr_out, tok_out, next_out, accepting_out);
    } catch (const std::bad_alloc&) {
        return fail(CD_ERR_OOM, "host allocation failed");
    } catch (...) {
        return fail(CD_ERR_INTERNAL, "unexpected exception");
    }
}

cd_status cd_compile_trie(int32_t V, int32_t K, const int64_t* label_ptr, const int32_t* label_tok, int32_t eos,
                          int device, cd_dfa_t** out) {
    try {
        if (!out || !label_ptr) return fail(CD_ERR_ARG, "NULL argument");
        if (V < 1 || K < 1) return fail(CD_ERR_ARG, "V and K must be >= 1");
        if (label_ptr[K] > 0 && !label_tok) return fail(CD_ERR_ARG, "label_tok is NULL");
        cdt::HostCsr c;
        const std::string err = cdt::build_trie(V, K, label_ptr, label_tok, eos, &c);
        if (!err.empty()) return fail(CD_ERR_AUTOMATON, "%s", err.c_str());
        return compile_csr(V, c, device, out);
    } catch (const std::bad_alloc&) {
        return fail(CD_ERR_OOM, "host allocation failed");
    } catch (...) {
        return fail(CD_ERR_INTERNAL, "unexpected exception");
    }
}

void cd_free_dfa(cd_dfa_t* d) {
    if (!d) return;
    DeviceGuard guard(d->device);
    for (auto& kv : d->scratch) kv.second.release();
    cudaFree(d->d_mask); cudaFree(d->d_row_ptr); cudaFree(d->d_tok); cudaFree(d->d_next); cudaFree(d->d_acc);
    cudaFree(d->d_rank); cudaFree(d->d_satisfying);
    delete d;
}

cd_status cd_dfa_info(const cd_dfa_t* d, int32_t* V, int32_t* S, int32_t* start, int64_t* nnz, int64_t* mask_bytes) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (V) *V = d->dev.V;
    if (S) *S = d->dev.S;
    if (start) *start = d->start;
    if (nnz) *nnz = d->nnz;
    if (mask_bytes) *mask_bytes = (int64_t)d->dev.S * d->dev.Wpad * 4;
    return CD_OK;
}

cd_status cd_set_gather_max(cd_dfa_t* d, int32_t max_transitions) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (max_transitions < -1) return fail(CD_ERR_ARG, "max_transitions must be >= -1");
    std::lock_guard<std::mutex> lk(d->mu);
    d->cfg.gather_max = max_transitions;
    return CD_OK;
}

cd_status cd_set_loop_mode(cd_dfa_t* d, int32_t mode) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (mode != CD_LOOP_AUTO && mode != CD_LOOP_PER_STEP && mode != CD_LOOP_BARRIER)
        return fail(CD_ERR_ARG, "mode must be CD_LOOP_AUTO, CD_LOOP_PER_STEP or CD_LOOP_BARRIER");
    std::lock_guard<std::mutex> lk(d->mu);
    d->cfg.loop_mode = mode;
    return CD_OK;
}

cd_status cd_reserve(const cd_dfa_t* d, int32_t max_rows, void* cuda_stream) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (max_rows < 0) return fail(CD_ERR_ARG, "max_rows < 0");
    DeviceGuard guard(d->device);
    Scratch* s = nullptr;
    return get_scratch(d, static_cast<cudaStream_t>(cuda_stream), max_rows, &s);
}

cd_status cd_step(const cd_dfa_t* d, const void* logits, cd_dtype dtype, int64_t ld_elems, const int32_t* row_map,
                  int32_t* state, int32_t n, int32_t* token_out, float* logprob_out, float* lse_out,
                  uint8_t* done_out, void* cuda_stream) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (n < 0) return fail(CD_ERR_ARG, "n < 0");
    cd_status st = check_dtype(dtype);
    if (st != CD_OK) return st;
    if (n == 0) return CD_OK;
    if (!state || !token_out || !logprob_out || !done_out) return fail(CD_ERR_ARG, "NULL output / state pointer");
    st = check_logits_layout(d, logits, dtype, ld_elems);
    if (st != CD_OK) return st;
    if ((long long)n * tiles_per_row(d->dev.V, dtype) >= 0x7FFFFFFFLL)
        return fail(CD_ERR_ARG, "n * tiles_per_row overflows the unit index");
    DeviceGuard guard(d->device);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const Settings cfg = settings_of(d);
    Scratch* s = nullptr;
    st = get_scratch(d, stream, n, &s);
    if (st != CD_OK) return st;
    return launch_step(d, cfg, s, logits, dtype, ld_elems, row_map, state, n, nullptr, token_out, logprob_out, lse_out,
                       done_out, stream);
}

cd_status cd_transition(const cd_dfa_t* d, const int32_t* token, int32_t* state, int32_t n, uint8_t* done_out,
                        void* cuda_stream) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (n < 0) return fail(CD_ERR_ARG, "n < 0");
    if (n == 0) return CD_OK;
    if (!token || !state || !done_out) return fail(CD_ERR_ARG, "NULL pointer");
    DeviceGuard guard(d->device);
    const int threads = 256;
    long long blocks = ((long long)n * 32 + threads - 1) / threads;
    if (blocks > 8192) blocks = 8192;
    cd::transition_kernel<<<(int)blocks, threads, 0, static_cast<cudaStream_t>(cuda_stream)>>>(d->dev, token, state, n,
                                                                                              done_out);
    CU(cudaGetLastError());
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return CD_OK;
}

cd_status cd_compact(const uint8_t* done, const int32_t* row_ids_in, const int32_t* state_in, int32_t n,
                     int32_t* row_ids_out, int32_t* state_out, int32_t* n_active_out, void* cuda_stream) {
    if (n < 0) return fail(CD_ERR_ARG, "n < 0");
    if (!n_active_out) return fail(CD_ERR_ARG, "n_active_out is NULL");
    if (n > 0 && (!done || !row_ids_out)) return fail(CD_ERR_ARG, "NULL pointer");
    if (n > 0 && state_in && !state_out) return fail(CD_ERR_ARG, "state_in given without state_out");
    return launch_compact(done, row_ids_in, state_in, n, row_ids_out, state_out, n_active_out, nullptr,
                          static_cast<cudaStream_t>(cuda_stream));
}

// cd_compact without any allocation: the scan's chunk words are the library's own fixed array (see above and cd.h).
cd_status cd_compact_noalloc(const uint8_t* done, const int32_t* row_ids_in, const int32_t* state_in, int32_t n,
                             int32_t* row_ids_out, int32_t* state_out, int32_t* n_active_out, void* cuda_stream) {
    if (n < 0) return fail(CD_ERR_ARG, "n < 0");
    if (n > CD_COMPACT_NOALLOC_MAX_N)
        return fail(CD_ERR_ARG, "cd_compact_noalloc: n = %d is above the fixed scratch of this entry point (at most %d slots per call); "
                    "split the list or use cd_compact", (int)n, (int)CD_COMPACT_NOALLOC_MAX_N);
    if (!n_active_out) return fail(CD_ERR_ARG, "n_active_out is NULL");
    if (n > 0 && (!done || !row_ids_out)) return fail(CD_ERR_ARG, "NULL pointer");
    if (n > 0 && state_in && !state_out) return fail(CD_ERR_ARG, "state_in given without state_out");
    return launch_compact_noalloc(done, row_ids_in, state_in, n, row_ids_out, state_out, n_active_out,
                                  static_cast<cudaStream_t>(cuda_stream));
}

static cd_status decode_loop_impl(const cd_dfa_t* d, const void* const* step_logits, cd_dtype dtype, int64_t ld_elems,
                                  int32_t B, int32_t max_steps, int32_t* tokens_out, int32_t* len_out,
                                  int32_t* final_state_out, float* sum_logprob_out, uint8_t* done_out,
                                  const LimitArgs& lim_in, void* cuda_stream, bool sync = true) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (B < 0 || max_steps < 0) return fail(CD_ERR_ARG, "B / max_steps < 0");
    const Settings cfg = settings_of(d);
    const LimitArgs lim = resolve_limit(cfg, lim_in);
    cd_status st = check_dtype(dtype);
    if (st != CD_OK) return st;
    if (B == 0) return CD_OK;
    if (!len_out || !final_state_out || !sum_logprob_out || !done_out || (max_steps > 0 && !tokens_out))
        return fail(CD_ERR_ARG, "NULL output pointer");
    if (max_steps > 0 && !step_logits) return fail(CD_ERR_ARG, "step_logits is NULL");
    if (!d->start_accepting)
        for (int k = 0; k < max_steps; ++k) {
            st = check_logits_layout(d, step_logits[k], dtype, ld_elems);
            if (st != CD_OK) return st;
        }
    RangeGuard range("cd_decode_loop");
    DeviceGuard guard(d->device);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    Scratch* s = nullptr;
    st = get_scratch(d, stream, B, &s);
    if (st != CD_OK) return st;
    bool persist = persistent_loop_possible(d, cfg, B, max_steps);
    // no LIMIT: the barrier-free kernel (every row advances through its steps independently); with a LIMIT, or
    // on request, the lock-step kernel (a LIMIT is defined step by step over ALL rows)
    if (persist && !lim.sat_ctr && cfg.loop_mode != CD_LOOP_BARRIER && flow_loop_possible(d, B, max_steps, dtype)) {
        st = enqueue_flow_loop(d, cfg, s, step_logits, dtype, ld_elems, B, max_steps, tokens_out, len_out,
                               final_state_out, sum_logprob_out, done_out, stream);
        if (st != CD_OK) return st;
        return sync ? finish_flow_loop(s, stream) : CD_OK;
    }
    if (!sync) persist = false;  // a lock-step loop holds the device's cooperative-launch lock until it has finished
    // Two lock-step loops must never share the SMs: each waits at its grid barrier for CTAs that the other
    // one keeps from being scheduled.  Within this process they are serialised per device (the loop
    // synchronises its stream before returning anyway).
    std::unique_lock<std::mutex> coop_lock;
    if (persist) {
        coop_lock = std::unique_lock<std::mutex>(coop_mutex(d->device));
        st = get_loop_scratch(s, max_steps, stream);
        if (st != CD_OK) return st;
        // both forms of the set-up are cheap; the persistent one is tried first and tells whether its CTAs fit
        st = launch_loop_init(d, s, B, max_steps, tokens_out, len_out, final_state_out, sum_logprob_out, done_out,
                              stream, lim, true);
        if (st != CD_OK) return st;
        bool launched = false;
        st = enqueue_persistent_loop(d, cfg, s, step_logits, dtype, ld_elems, B, max_steps, tokens_out, len_out,
                                     final_state_out, sum_logprob_out, done_out, stream, lim, &launched);
        if (st != CD_OK) return st;
        persist = launched;
    }
    if (!persist) {
        st = launch_loop_init(d, s, B, max_steps, tokens_out, len_out, final_state_out, sum_logprob_out, done_out,
                              stream, lim);
        if (st != CD_OK) return st;
        if (!d->start_accepting)
            for (int k = 0; k < max_steps; ++k) {
                st = enqueue_loop_step(d, cfg, s, step_logits[k], dtype, ld_elems, B, k, max_steps, tokens_out, len_out,
                                       final_state_out, sum_logprob_out, done_out, stream, lim);
                if (st != CD_OK) return st;
            }
    }
    if (!sync) {  // the loop's error count joins the status word cd_loop_sync reads
        st = get_status_word(s);
        if (st != CD_OK) return st;
        cd::fold_status_kernel<<<1, 1, 0, stream>>>(s->b.ctrs, s->d_status);
        CU(cudaGetLastError());
        g_launches.fetch_add(1, std::memory_order_relaxed);
        return CD_OK;
    }
    return finish_loop(s, stream, persist);
}

cd_status cd_decode_loop_async(const cd_dfa_t* d, const void* const* step_logits, cd_dtype dtype, int64_t ld_elems,
                               int32_t B, int32_t max_steps, int32_t* tokens_out, int32_t* len_out,
                               int32_t* final_state_out, float* sum_logprob_out, uint8_t* done_out, void* cuda_stream) {
    return decode_loop_impl(d, step_logits, dtype, ld_elems, B, max_steps, tokens_out, len_out, final_state_out,
                            sum_logprob_out, done_out, LimitArgs(), cuda_stream, false);
}

cd_status cd_loop_sync(const cd_dfa_t* d, void* cuda_stream) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    DeviceGuard guard(d->device);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    cd_dfa* dm = const_cast<cd_dfa*>(d);
    Scratch* s = nullptr;
    {
        std::lock_guard<std::mutex> lk(dm->mu);
        auto it = dm->scratch.find(stream);
        if (it != dm->scratch.end()) s = &it->second;
    }
    if (!s) {
        CU(cudaStreamSynchronize(stream));
        return CD_OK;
    }
    return finish_flow_loop(s, stream);
}

cd_status cd_decode_loop(const cd_dfa_t* d, const void* const* step_logits, cd_dtype dtype, int64_t ld_elems,
                         int32_t B, int32_t max_steps, int32_t* tokens_out, int32_t* len_out,
                         int32_t* final_state_out, float* sum_logprob_out, uint8_t* done_out, void* cuda_stream) {
    return decode_loop_impl(d, step_logits, dtype, ld_elems, B, max_steps, tokens_out, len_out, final_state_out,
                            sum_logprob_out, done_out, LimitArgs(), cuda_stream);
}

cd_status cd_loop_trace(const cd_dfa_t* d, void* cuda_stream, int32_t cap, int64_t* t_ns_out, int32_t* n_active_out,
                        int32_t* steps_out) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (cap < 0 || !steps_out || (cap > 0 && (!t_ns_out || !n_active_out))) return fail(CD_ERR_ARG, "bad argument");
    DeviceGuard guard(d->device);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    cd_dfa* dm = const_cast<cd_dfa*>(d);
    *steps_out = 0;
    const unsigned long long* tt = nullptr;
    const int* tn = nullptr;
    const int* f_q = nullptr;  // flow_kernel: which of its two buffer pairs is told by the launch counter's parity
    const unsigned long long* ftt[2] = {nullptr, nullptr};
    const int* ftn[2] = {nullptr, nullptr};
    {  // only the pointers are taken under the handle's lock: other threads using the handle do not wait for this stream
        std::lock_guard<std::mutex> lk(dm->mu);
        auto it = dm->scratch.find(stream);
        if (it != dm->scratch.end() && it->second.trace_src == 1) {
            tt = it->second.b.trace_t;
            tn = it->second.b.trace_n;
        } else if (it != dm->scratch.end() && it->second.trace_src == 2) {
            f_q = it->second.b.f_q;
            for (int i = 0; i < 2; ++i) {
                ftt[i] = it->second.b.f_trace_t[i];
                ftn[i] = it->second.b.f_trace_n[i];
            }
        }
    }
    if (f_q) {  // the buffers of the last launch are the ones the launch counter's parity no longer names
        int par = 0;
        CU(cudaMemcpyAsync(&par, f_q + cd::FQ_LAUNCHES, sizeof(int), cudaMemcpyDeviceToHost, stream));
        CU(cudaStreamSynchronize(stream));
        tt = ftt[(par & 1) ^ 1];
        tn = ftn[(par & 1) ^ 1];
    }
    if (!tt) return CD_OK;  // the last loop on this stream did not run in a persistent kernel
    std::vector<unsigned long long> ht((size_t)cd::LOOP_TRACE_STEPS + 1);
    std::vector<int> hn((size_t)cd::LOOP_TRACE_STEPS + 1);
    CU(cudaMemcpyAsync(ht.data(), tt, sizeof(unsigned long long) * ht.size(), cudaMemcpyDeviceToHost, stream));
    CU(cudaMemcpyAsync(hn.data(), tn, sizeof(int) * hn.size(), cudaMemcpyDeviceToHost, stream));
    CU(cudaStreamSynchronize(stream));
    int steps = hn[cd::LOOP_TRACE_STEPS];
    if (steps > cd::LOOP_TRACE_STEPS) steps = cd::LOOP_TRACE_STEPS;
    *steps_out = steps;
    // (row tasks: entry k is the latest publication of a task of step k -- keep the times monotone)
    for (int k = 1; k <= steps; ++k)
        if (ht[(size_t)k] < ht[(size_t)k - 1]) ht[(size_t)k] = ht[(size_t)k - 1];
    for (int k = 0; k < steps && k < cap; ++k) {
        n_active_out[k] = hn[(size_t)k];
        t_ns_out[k] = (int64_t)(ht[(size_t)k + 1] - ht[(size_t)k]);
    }
    return CD_OK;
}

#ifdef CD_TUNING
// tuning builds only (not declared in cd.h): the raw phase timestamps of the last persistent loop
__attribute__((visibility("default"))) cd_status cd_loop_phase_trace(const cd_dfa_t* d, void* cuda_stream, uint64_t* out /*[256][8]*/,
                                                                      uint64_t* t_out /*[257]*/) {
    DeviceGuard guard(d->device);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    cd_dfa* dm = const_cast<cd_dfa*>(d);
    Scratch* s = nullptr;
    {
        std::lock_guard<std::mutex> lk(dm->mu);
        s = &dm->scratch[stream];
    }
    CU(cudaMemcpyAsync(out, s->b.phase, sizeof(uint64_t) * (size_t)cd::LOOP_TRACE_STEPS * 8, cudaMemcpyDeviceToHost, stream));
    CU(cudaMemcpyAsync(t_out, s->b.trace_t, sizeof(uint64_t) * ((size_t)cd::LOOP_TRACE_STEPS + 1), cudaMemcpyDeviceToHost, stream));
    CU(cudaStreamSynchronize(stream));
    return CD_OK;
}
#endif

cd_status cd_set_satisfying(cd_dfa_t* d, const uint8_t* satisfying) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    DeviceGuard guard(d->device);
    std::lock_guard<std::mutex> lk(d->mu);
    if (!satisfying) {
        d->cfg.has_satisfying = false;  // the device array stays allocated: a loop in flight may still read it
        return CD_OK;
    }
    CU(cudaMemcpy(d->d_satisfying, satisfying, (size_t)d->dev.S, cudaMemcpyHostToDevice));
    d->cfg.has_satisfying = true;
    return CD_OK;
}

cd_status cd_decode_loop_limit(const cd_dfa_t* d, const void* const* step_logits, cd_dtype dtype, int64_t ld_elems,
                               int32_t B, int32_t max_steps, int32_t* tokens_out, int32_t* len_out,
                               int32_t* final_state_out, float* sum_logprob_out, uint8_t* done_out, int32_t limit,
                               int32_t* satisfied_inout, void* cuda_stream) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (!settings_of(d).has_satisfying) return fail(CD_ERR_ARG, "cd_set_satisfying has not been called on this automaton");
    if (!satisfied_inout) return fail(CD_ERR_ARG, "satisfied_inout is NULL");
    if (limit < 0) return fail(CD_ERR_ARG, "limit < 0");
    LimitArgs lim;
    lim.sat_ctr = satisfied_inout;
    lim.limit = limit;
    return decode_loop_impl(d, step_logits, dtype, ld_elems, B, max_steps, tokens_out, len_out, final_state_out,
                            sum_logprob_out, done_out, lim, cuda_stream);
}

cd_status cd_decode_loop_host(const cd_dfa_t* d, const void* const* step_logits_host, cd_dtype dtype,
                              int64_t ld_elems, int32_t B, int32_t max_steps, int32_t* tokens_out, int32_t* len_out,
                              int32_t* final_state_out, float* sum_logprob_out, uint8_t* done_out,
                              void* cuda_stream) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (B < 0 || max_steps < 0) return fail(CD_ERR_ARG, "B / max_steps < 0");
    cd_status st = check_dtype(dtype);
    if (st != CD_OK) return st;
    if (B == 0) return CD_OK;
    if (!len_out || !final_state_out || !sum_logprob_out || !done_out || (max_steps > 0 && !tokens_out))
        return fail(CD_ERR_ARG, "NULL output pointer");
    if (max_steps > 0 && !step_logits_host) return fail(CD_ERR_ARG, "step_logits_host is NULL");
    const long long sz = dtype == CD_BF16 ? 2 : 4;
    if (ld_elems < d->dev.V) return fail(CD_ERR_ARG, "ld_elems < V");
    if ((ld_elems * sz) % 16 != 0) return fail(CD_ERR_ARG, "row stride is not a multiple of 16 bytes");
    for (int k = 0; k < max_steps; ++k)
        if (!step_logits_host[k]) return fail(CD_ERR_ARG, "step_logits_host[%d] is NULL", k);

    RangeGuard range("cd_decode_loop_host");
    DeviceGuard guard(d->device);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const Settings cfg = settings_of(d);
    Scratch* s = nullptr;
    st = get_scratch(d, stream, B, &s);
    if (st != CD_OK) return st;

    // one staging buffer (the active rows of one step, compact) + device copies of the outputs
    const size_t step_bytes = (size_t)B * (size_t)ld_elems * (size_t)sz;
    const size_t n_tok = (size_t)B * (size_t)(max_steps > 0 ? max_steps : 1);
    const size_t out_bytes = sizeof(int) * (n_tok + 3 * (size_t)B) + (size_t)B + 64;
    st = get_host_loop_scratch(s, step_bytes, 0, out_bytes, stream);
    if (st != CD_OK) return st;
    int* d_tokens = s->out_i32;
    int* d_len = d_tokens + n_tok;
    int* d_fs = d_len + B;
    float* d_slp = reinterpret_cast<float*>(d_fs + B);
    uint8_t* d_done = reinterpret_cast<uint8_t*>(d_slp + B);

    const LimitArgs lim = resolve_limit(cfg);
    st = launch_loop_init(d, s, B, max_steps, d_tokens, d_len, d_fs, d_slp, d_done, stream, lim);
    if (st != CD_OK) return st;
    if (!d->start_accepting && max_steps > 0) {
        // Pinned, device-mapped host buffers (what cudaHostAlloc / torch pin_memory give under unified
        // addressing): the SMs pull the active rows over PCIe themselves, nothing is read back per step.
        bool mapped = tune_int("CD_HOST_ZEROCOPY", 1, 0, 1) != 0;
        std::vector<const unsigned char*> dev_view((size_t)max_steps, nullptr);
        for (int k = 0; k < max_steps && mapped; ++k) {
            cudaPointerAttributes at;
            if (cudaPointerGetAttributes(&at, step_logits_host[k]) != cudaSuccess) {
                cudaGetLastError();
                mapped = false;
            } else if (at.type != cudaMemoryTypeHost || !at.devicePointer ||
                       (reinterpret_cast<uintptr_t>(at.devicePointer) & 15) != 0) {
                mapped = false;
            } else {
                dev_view[(size_t)k] = static_cast<const unsigned char*>(at.devicePointer);
            }
        }
        // Density-adaptive step over PCIe (cd_set_gather_max != 0): a masked log-softmax needs only
        // the allowed logits, and over a 51 GB/s link that is where it pays most.  When EVERY state may be
        // gathered, the step kernel reads the allowed logits of the active rows straight from the mapped host
        // buffer (one 32-byte sector each) and nothing is staged: configs[4] moves 42 KB per row-step instead
        // of 512 KB.  Threshold: the caller's, or automatic = V / 32 transitions (a gathered logit costs a
        // 32-byte sector on the link against 2 or 4 bytes per token of a full row; half the break-even).
        const long long host_gmax = cfg.gather_max > 0 ? cfg.gather_max : (cfg.gather_max < 0 ? d->dev.V / 32 : 0);
        if (mapped && host_gmax > 0 && d->max_deg <= host_gmax) {
            Settings gcfg = cfg;
            gcfg.gather_max = (int)std::min<long long>(host_gmax, 0x3FFFFFFF);
            for (int k = 0; k < max_steps; ++k) {
                st = enqueue_loop_step(d, gcfg, s, dev_view[(size_t)k], dtype, ld_elems, B, k, max_steps, d_tokens, d_len, d_fs,
                                       d_slp, d_done, stream, lim, 0);
                if (st != CD_OK) return st;
            }
        } else if (mapped) {
            const unsigned long long row_bytes = (unsigned long long)ld_elems * (unsigned long long)sz;
            for (int k = 0; k < max_steps; ++k) {
                const int cur = k & 1;
                cd::host_gather_rows_kernel<<<d->num_sms * host_gather_mult(), 256, 0, stream>>>(
                    dev_view[(size_t)k], row_bytes, s->b.row_ids[cur], s->b.n_active + cur,
                    static_cast<unsigned char*>(s->stage[0]));
                CU(cudaGetLastError());
                g_launches.fetch_add(1, std::memory_order_relaxed);
                st = enqueue_loop_step(d, cfg, s, s->stage[0], dtype, ld_elems, B, k, max_steps, d_tokens, d_len, d_fs,
                                       d_slp, d_done, stream, lim, 1);
                if (st != CD_OK) return st;
            }
        } else {
            // Early exit reaches the PCIe link too: only the rows still active are copied.  After step
            // k - 1 the host reads the compacted active list (n and the original row ids), copies those
            // rows of step k's logits into the compact staging buffer (runs of consecutive ids as one copy)
            // and launches the step with logits row = slot.  Kernel time is ~1 % of the copy time, so
            // nothing is lost by not overlapping the two.
            if (s->h_ids_cap < B) {
                if (s->h_ids) cudaFreeHost(s->h_ids);
                s->h_ids = nullptr;
                s->h_ids_cap = 0;
                CU(cudaMallocHost(&s->h_ids, sizeof(int) * (size_t)B));
                s->h_ids_cap = B;
            }
            const size_t row_bytes = (size_t)ld_elems * (size_t)sz;
            int n_h = B;
            for (int i = 0; i < B; ++i) s->h_ids[i] = i;
            for (int k = 0; k < max_steps; ++k) {
                const int cur = k & 1;
                if (k > 0 || lim.sat_ctr) {  // (with a LIMIT the list may be empty from the start)
                    CU(cudaMemcpyAsync(s->h_pinned, s->b.n_active + cur, sizeof(int), cudaMemcpyDeviceToHost, stream));
                    CU(cudaMemcpyAsync(s->h_ids, s->b.row_ids[cur], sizeof(int) * (size_t)B, cudaMemcpyDeviceToHost, stream));
                    CU(cudaStreamSynchronize(stream));
                    n_h = s->h_pinned[0];
                }
                if (n_h <= 0) break;
                const unsigned char* src = static_cast<const unsigned char*>(step_logits_host[k]);
                unsigned char* dst = static_cast<unsigned char*>(s->stage[0]);
                for (int i = 0; i < n_h;) {
                    int e = i + 1;
                    while (e < n_h && s->h_ids[e] == s->h_ids[e - 1] + 1) ++e;
                    CU(cudaMemcpyAsync(dst + (size_t)i * row_bytes, src + (size_t)s->h_ids[i] * row_bytes,
                                       (size_t)(e - i) * row_bytes, cudaMemcpyHostToDevice, stream));
                    i = e;
                }
                st = enqueue_loop_step(d, cfg, s, s->stage[0], dtype, ld_elems, B, k, max_steps, d_tokens, d_len, d_fs,
                                       d_slp, d_done, stream, lim, 1);
                if (st != CD_OK) return st;
            }
        }
    }
    if (max_steps > 0)
        CU(cudaMemcpyAsync(tokens_out, d_tokens, sizeof(int) * (size_t)B * max_steps, cudaMemcpyDeviceToHost, stream));
    CU(cudaMemcpyAsync(len_out, d_len, sizeof(int) * (size_t)B, cudaMemcpyDeviceToHost, stream));
    CU(cudaMemcpyAsync(final_state_out, d_fs, sizeof(int) * (size_t)B, cudaMemcpyDeviceToHost, stream));
    CU(cudaMemcpyAsync(sum_logprob_out, d_slp, sizeof(float) * (size_t)B, cudaMemcpyDeviceToHost, stream));
    CU(cudaMemcpyAsync(done_out, d_done, (size_t)B, cudaMemcpyDeviceToHost, stream));
    return finish_loop(s, stream, false);
}

}  // extern "C"

// =============================================================================== LM-head step
namespace {

using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess)
            p = nullptr;
        return reinterpret_cast<EncodeTiledFn>(p);
    }();
    return fn;
}

// bf16 [rows, ld] row-major, box = box_rows x 64 elements (128 bytes), 128-byte swizzle, OOB -> 0
cd_status make_tmap_bf16(CUtensorMap* out, const void* base, long long rows, long long cols, long long ld,
                         int box_rows) {
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return fail(CD_ERR_CUDA, "cuTensorMapEncodeTiled is not available from this driver");
    const cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)ld * 2};
    const cuuint32_t box[2] = {(cuuint32_t)cd::HD_BK, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(CD_ERR_CUDA, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
    return CD_OK;
}

// Launch with programmatic stream serialization (as launch_step_t): the kernels of an LM-head step are short and
// many (prepare, gather, gather finish, pack, two contractions of which one returns at once, finish, loop tail);
// each begins with griddepcontrol.wait, so the next one's launch overlaps the running one instead of following it.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kern)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t stream, Args&&... args) {
    cudaLaunchConfig_t lc{};
    lc.gridDim = dim3(grid);
    lc.blockDim = dim3(block);
    lc.dynamicSmemBytes = smem;
    lc.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = use_pdl() ? 1 : 0;
    lc.attrs = at;
    lc.numAttrs = 1;
    return cudaLaunchKernelEx(&lc, kern, std::forward<Args>(args)...);
}

cd_status get_head_scratch(Scratch* s, int rows, int H, cudaStream_t stream) {
    if (s->head_rows >= rows && s->head_H == H) return CD_OK;  // the A tensor map is built for exactly H columns
    if (s->head_rows > 0) CU(cudaStreamSynchronize(stream));
    s->release_head();
    if (rows < s->b.cap_rows) rows = s->b.cap_rows;
    const long long rows_pad = ((long long)rows + cd::HD_BM - 1) / cd::HD_BM * cd::HD_BM;
    const long long ldA = ((long long)H + 7) / 8 * 8;
    cudaError_t e = cudaSuccess;
    auto A = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
    A(cudaMalloc(&s->h_flags, (size_t)rows * 2));
    A(cudaMalloc(&s->h_lists, sizeof(int) * (size_t)rows * 4));
    A(cudaMalloc(&s->h_ctr, sizeof(int) * 4));
    A(cudaMalloc(&s->h_A, (size_t)rows_pad * (size_t)ldA * 2));
    A(cudaMalloc(&s->h_partials, sizeof(cd::HeadPartial) * (size_t)cd::head_partials_cap(rows)));
    A(cudaMalloc(&s->h_gpartials, sizeof(cd::HeadPartial) * (size_t)rows * cd::HG_MAX_PIECES));
    if (e == cudaSuccess) e = cudaMemset(s->h_ctr, 0, sizeof(int) * 4);
    if (e == cudaSuccess) e = cudaMemset(s->h_A, 0, (size_t)rows_pad * (size_t)ldA * 2);
    cd_status st = CD_OK;
    if (e != cudaSuccess)
        st = fail(e == cudaErrorMemoryAllocation ? CD_ERR_OOM : CD_ERR_CUDA, "LM-head scratch: %s", cudaGetErrorString(e));
    s->h_ldA = ldA;
    if (st == CD_OK) st = make_tmap_bf16(&s->h_tmA, s->h_A, rows_pad, H, ldA, cd::HD_BM);
    if (st != CD_OK) {
        s->release_head();  // nothing half-built is kept
        return st;
    }
    s->head_rows = rows;
    s->head_H = H;
    return CD_OK;
}

// Largest number of transitions a state may have for its rows to be gathered by the LM-head
// step.  A gathered logit reads one W row (2H bytes, mostly from L2) and costs 2H flops on the
// CUDA cores; a dense row costs 2VH flops on the tensor cores.  Automatic policy: gather while
// deg * 2H bytes at ~4 TB/s is below V * 2H flops at ~1.2 PFLOP/s, i.e. deg < V / 300.
int head_gather_max_for(const cd_dfa* d, const Settings& cfg) {
    if (cfg.head_gather_max >= 0) return cfg.head_gather_max;
    return d->dev.V / 300 > 1 ? d->dev.V / 300 : 1;
}

cd_status check_head_layout(const void* hidden, long long ldh, const void* W, long long ldw, int H) {
    if (H < 8 || (H % 8) != 0) return fail(CD_ERR_ARG, "H (%d) must be a positive multiple of 8", H);
    if (!hidden || !W) return fail(CD_ERR_ARG, "hidden / W is NULL");
    if (ldh < H || ldw < H) return fail(CD_ERR_ARG, "ldh_elems / ldw_elems < H");
    if ((ldh % 8) != 0 || (ldw % 8) != 0) return fail(CD_ERR_ARG, "row strides must be multiples of 8 elements (16 bytes)");
    if ((reinterpret_cast<uintptr_t>(hidden) & 15) != 0 || (reinterpret_cast<uintptr_t>(W) & 15) != 0)
        return fail(CD_ERR_ARG, "hidden / W base is not 16-byte aligned");
    if ((size_t)H * 2 > 200 * 1024) return fail(CD_ERR_ARG, "H too large (hidden row must fit in shared memory)");
    return CD_OK;
}

// tensor map of the output embedding, cached per handle (the weights rarely change)
cd_status head_weight_map(const cd_dfa* d, const void* W, long long ldw, int H, CUtensorMap* out, CUtensorMap* out_half) {
    cd_dfa* dm = const_cast<cd_dfa*>(d);
    std::lock_guard<std::mutex> lk(dm->mu);
    if (dm->w_ptr != W || dm->w_ld != ldw || dm->w_H != H) {
        cd_status st = make_tmap_bf16(&dm->w_tmap, W, d->dev.V, H, ldw, cd::HD_BN);
        if (st == CD_OK) st = make_tmap_bf16(&dm->w_tmap_half, W, d->dev.V, H, ldw, cd::HD2_HALF_N);
        if (st != CD_OK) {
            dm->w_ptr = nullptr;
            return st;
        }
        dm->w_ptr = W; dm->w_ld = ldw; dm->w_H = H;
    }
    *out = dm->w_tmap;  // copied under the lock: concurrent callers may use different weights
    *out_half = dm->w_tmap_half;
    return CD_OK;
}

// The kernels of one LM-head step for up to n_upper active slots (n_dev overrides the count on
// the device).  With loop extras the rows' history is recorded as they finalise and a last
// one-CTA kernel compacts the active list.
cd_status launch_head(const cd_dfa* d, const Settings& cfg, Scratch* s, const void* hidden, long long ldh, const void* W, long long ldw, int H,
                      const int* row_map, int* state, int n_upper, const int* n_dev, int* token_out, float* logprob_out,
                      float* lse_out, uint8_t* done_out, cudaStream_t stream, const LoopExtras* x) {
    cd::HeadArgs a{};
    if (x) {
        a.fin.hist_tokens = x->tokens;
        a.fin.hist_len = x->len;
        a.fin.hist_final_state = x->final_state;
        a.fin.hist_sum_logprob = x->sum_logprob;
        a.fin.hist_done = x->done;
        a.fin.step = x->step;
        a.fin.max_steps = x->max_steps;
        a.fin.cmp_row_ids_out = x->row_ids_out;
        a.fin.cmp_state_out = x->state_out;
        a.fin.cmp_n_out = x->n_out;
        a.fin.logits_by_slot = x->logits_by_slot;  // here: hidden rows indexed by slot
        a.fin.satisfying = x->satisfying;
        a.fin.sat_ctr = x->sat_ctr;
        a.fin.limit = x->limit;
    }
    a.fin.dfa = d->dev;
    a.fin.row_map = row_map;
    a.fin.state = state;
    a.fin.state_new = state;
    a.fin.n = n_upper;
    a.fin.n_dev = n_dev;
    a.fin.token_out = token_out;
    a.fin.logprob_out = logprob_out;
    a.fin.lse_out = lse_out;
    a.fin.done_out = done_out;
    a.fin.ctrs = s->b.ctrs;
    a.fin.inv_tau = cfg.inv_tau;
    a.fin.seed_lo = (uint32_t)(cfg.seed & 0xFFFFFFFFull);
    a.fin.seed_hi = (uint32_t)(cfg.seed >> 32);
    a.fin.rng_step_base = cfg.rng_step_base;
    const bool sample = cfg.inv_tau > 0.0f;
    a.hidden = static_cast<const uint16_t*>(hidden);
    a.ldh = ldh;
    a.W = static_cast<const uint16_t*>(W);
    a.ldw = ldw;
    a.H = H;
    a.gather_max = head_gather_max_for(d, cfg);
    a.gather_auto = (cfg.head_gather_max < 0) ? 1 : 0;
    {  // most pieces a gathered row can have: the automatic policy may gather any state
        const long long gdeg = a.gather_auto ? d->max_deg : std::min<long long>(d->max_deg, a.gather_max);
        a.gp_max = cd::hg_pieces((int)std::min<long long>(gdeg, 0x7FFFFFFF));
    }
    a.gpartials = s->h_gpartials;
    a.not_dense = s->h_flags;
    a.not_gather = s->h_flags + s->head_rows;
    a.dense_slot = s->h_lists;
    a.dense_state = s->h_lists + s->head_rows;
    a.gather_slot = s->h_lists + 2 * (size_t)s->head_rows;
    a.gather_state = s->h_lists + 3 * (size_t)s->head_rows;
    a.hctr = s->h_ctr;
    a.A = s->h_A;
    a.ldA = s->h_ldA;
    a.partials = s->h_partials;

    const int n = n_upper;
    CUtensorMap tmW, tmWh;
    {
        const cd_status stw = head_weight_map(d, W, ldw, H, &tmW, &tmWh);
        if (stw != CD_OK) return stw;
    }
    // CTA pairs (thread-block clusters of 2) for calls with more than one row tile: needs an even number of SMs in
    // the grid and a batch that can have > 128 dense rows at all
    a.pairs = (head_pairs_enabled() && (d->num_sms % 2) == 0 && n_upper >= cd::HD2_MIN_ROWS) ? 1 : 0;
    CU(launch_pdl(cd::head_prepare_kernel, (unsigned)(1), (unsigned)(1024), (size_t)(0), stream, a));
    CU(cudaGetLastError());
    const bool any_gather = (a.gather_max > 0 && d->min_deg_nonacc <= a.gather_max) || (a.gather_auto && d->max_deg > a.gather_max);
    const bool any_dense = d->max_deg > a.gather_max;
    int launches = 1;
    if (any_gather) {
        const size_t smem = (size_t)H * 2;
        static thread_local int cfg_dev = -1;
        if (smem > 48 * 1024 && cfg_dev != d->device) {
            CU(cudaFuncSetAttribute(cd::head_gather_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
            CU(cudaFuncSetAttribute(cd::head_gather_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
            CU(cudaFuncSetAttribute(cd::head_gather_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
            CU(cudaFuncSetAttribute(cd::head_gather_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
            cfg_dev = d->device;
        }
        // one CTA per (row, piece), grid-stride: enough CTAs to fill the machine, never more than there are items
        long long gblocks = (long long)n * a.gp_max;
        if (gblocks > (long long)d->num_sms * 8) gblocks = (long long)d->num_sms * 8;
        const bool two = a.gp_max > 1;  // long rows (cut into pieces): two W rows per warp in flight
        if (sample) {
            if (two) CU(launch_pdl(cd::head_gather_kernel<true, true>, (unsigned)((int)gblocks), (unsigned)(cd::HG_WARPS * 32), (size_t)(smem), stream, a));
            else CU(launch_pdl(cd::head_gather_kernel<true, false>, (unsigned)((int)gblocks), (unsigned)(cd::HG_WARPS * 32), (size_t)(smem), stream, a));
        } else {
            if (two) CU(launch_pdl(cd::head_gather_kernel<false, true>, (unsigned)((int)gblocks), (unsigned)(cd::HG_WARPS * 32), (size_t)(smem), stream, a));
            else CU(launch_pdl(cd::head_gather_kernel<false, false>, (unsigned)((int)gblocks), (unsigned)(cd::HG_WARPS * 32), (size_t)(smem), stream, a));
        }
        CU(cudaGetLastError());
        ++launches;
        if (a.gp_max > 1) {  // rows cut into several pieces are merged and finished here
            const int fb = (n + 7) / 8;
            if (sample) CU(launch_pdl(cd::head_gather_finish_kernel<true>, (unsigned)(fb), (unsigned)(256), (size_t)(0), stream, a));
            else CU(launch_pdl(cd::head_gather_finish_kernel<false>, (unsigned)(fb), (unsigned)(256), (size_t)(0), stream, a));
            CU(cudaGetLastError());
            ++launches;
        }
    }
    if (any_dense) {
        const int rows_per_block = 8;
        CU(launch_pdl(cd::head_pack_kernel, (unsigned)((n + rows_per_block - 1) / rows_per_block), (unsigned)(rows_per_block * 32), (size_t)(0), stream, a));
        CU(cudaGetLastError());
        static thread_local int cfg_dev2 = -1;
        if (cfg_dev2 != d->device) {
            CU(cudaFuncSetAttribute(cd::head_dense_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, cd::HD_SMEM_BYTES));
            CU(cudaFuncSetAttribute(cd::head_dense_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, cd::HD_SMEM_BYTES));
            cfg_dev2 = d->device;
        }
        const int fin_blocks = (n + rows_per_block - 1) / rows_per_block;
        if (a.pairs) {
            static thread_local int cfg_dev3 = -1;
            if (cfg_dev3 != d->device) {
                CU(cudaFuncSetAttribute(cd::head_dense2_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, cd::HD2_SMEM_BYTES));
                CU(cudaFuncSetAttribute(cd::head_dense2_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, cd::HD2_SMEM_BYTES));
                cfg_dev3 = d->device;
            }
            // (the kernel carries __cluster_dims__(2, 1, 1); each of the two dense kernels returns at once when the
            // number of dense rows, known on the device only, puts the call in the other one's range)
            if (sample) CU(launch_pdl(cd::head_dense2_kernel<true>, (unsigned)(d->num_sms), (unsigned)(cd::HD_THREADS), (size_t)(cd::HD2_SMEM_BYTES), stream, s->h_tmA, tmWh, a));
            else CU(launch_pdl(cd::head_dense2_kernel<false>, (unsigned)(d->num_sms), (unsigned)(cd::HD_THREADS), (size_t)(cd::HD2_SMEM_BYTES), stream, s->h_tmA, tmWh, a));
            CU(cudaGetLastError());
            ++launches;
        }
        if (sample) {
            CU(launch_pdl(cd::head_dense_kernel<true>, (unsigned)(d->num_sms), (unsigned)(cd::HD_THREADS), (size_t)(cd::HD_SMEM_BYTES), stream, s->h_tmA, tmW, a));
            CU(cudaGetLastError());
            CU(launch_pdl(cd::head_finish_kernel<true>, (unsigned)(fin_blocks), (unsigned)(rows_per_block * 32), (size_t)(0), stream, a));
        } else {
            CU(launch_pdl(cd::head_dense_kernel<false>, (unsigned)(d->num_sms), (unsigned)(cd::HD_THREADS), (size_t)(cd::HD_SMEM_BYTES), stream, s->h_tmA, tmW, a));
            CU(cudaGetLastError());
            CU(launch_pdl(cd::head_finish_kernel<false>, (unsigned)(fin_blocks), (unsigned)(rows_per_block * 32), (size_t)(0), stream, a));
        }
        CU(cudaGetLastError());
        launches += 3;
    }
    if (x) {
        CU(launch_pdl(cd::head_loop_tail_kernel, (unsigned)(1), (unsigned)(1024), (size_t)(0), stream, a));
        CU(cudaGetLastError());
        ++launches;
    }
    g_launches.fetch_add(launches, std::memory_order_relaxed);
    return CD_OK;
}

}  // namespace

extern "C" {

cd_status cd_set_limit(cd_dfa_t* d, int32_t limit, int32_t* satisfied_inout) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    std::lock_guard<std::mutex> lk(d->mu);
    if (!satisfied_inout) {  // clear
        d->cfg.limit_ctr = nullptr;
        d->cfg.limit = 0;
        return CD_OK;
    }
    if (limit < 0) return fail(CD_ERR_ARG, "limit < 0");
    if (!d->cfg.has_satisfying) return fail(CD_ERR_ARG, "cd_set_satisfying has not been called on this automaton");
    d->cfg.limit_ctr = satisfied_inout;
    d->cfg.limit = limit;
    return CD_OK;
}

cd_status cd_set_sampling(cd_dfa_t* d, float temperature, uint64_t seed, int32_t step_base) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (!(temperature >= 0.0f) || temperature > 3.0e38f) return fail(CD_ERR_ARG, "temperature must be finite and >= 0");
    if (step_base < 0) return fail(CD_ERR_ARG, "step_base < 0");
    std::lock_guard<std::mutex> lk(d->mu);
    d->cfg.inv_tau = temperature > 0.0f ? 1.0f / temperature : 0.0f;  // IEEE fp32 division, as the oracle's
    d->cfg.seed = seed;
    d->cfg.rng_step_base = step_base;
    return CD_OK;
}

cd_status cd_set_head_gather_max(cd_dfa_t* d, int32_t max_transitions) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (max_transitions < -1) return fail(CD_ERR_ARG, "max_transitions must be >= -1");
    std::lock_guard<std::mutex> lk(d->mu);
    d->cfg.head_gather_max = max_transitions;
    return CD_OK;
}

cd_status cd_head_step(const cd_dfa_t* d, const void* hidden, int64_t ldh_elems, const void* W, int64_t ldw_elems,
                       int32_t H, const int32_t* row_map, int32_t* state, int32_t n, int32_t* token_out,
                       float* logprob_out, float* lse_out, uint8_t* done_out, void* cuda_stream) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (n < 0) return fail(CD_ERR_ARG, "n < 0");
    cd_status st = check_head_layout(hidden, ldh_elems, W, ldw_elems, H);
    if (st != CD_OK) return st;
    if (n == 0) return CD_OK;
    if (!state || !token_out || !logprob_out || !done_out) return fail(CD_ERR_ARG, "NULL pointer");
    DeviceGuard guard(d->device);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const Settings cfg = settings_of(d);
    Scratch* s = nullptr;
    st = get_scratch(d, stream, n, &s);
    if (st != CD_OK) return st;
    st = get_head_scratch(s, n, H, stream);
    if (st != CD_OK) return st;
    return launch_head(d, cfg, s, hidden, ldh_elems, W, ldw_elems, H, row_map, state, n, nullptr, token_out, logprob_out,
                       lse_out, done_out, stream, nullptr);
}

// Shared by cd_head_decode_loop (DEVICE hidden states) and cd_head_decode_loop_host (HOST hidden
// states and outputs: the H2D copy of step k+1 overlaps the kernels of step k).
static cd_status head_loop_impl(const cd_dfa_t* d, const void* const* step_hidden, bool host, int64_t ldh_elems,
                                const void* W, int64_t ldw_elems, int32_t H, int32_t B, int32_t max_steps,
                                int32_t* tokens_out, int32_t* len_out, int32_t* final_state_out,
                                float* sum_logprob_out, uint8_t* done_out, void* cuda_stream) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (B < 0 || max_steps < 0) return fail(CD_ERR_ARG, "B / max_steps < 0");
    if (B == 0) return CD_OK;
    if (!len_out || !final_state_out || !sum_logprob_out || !done_out || (max_steps > 0 && !tokens_out))
        return fail(CD_ERR_ARG, "NULL output pointer");
    if (max_steps > 0 && !step_hidden) return fail(CD_ERR_ARG, "step_hidden is NULL");
    cd_status st = CD_OK;
    for (int k = 0; k < max_steps; ++k) {
        // host rows need no 16-byte alignment of their own: they are copied into aligned staging
        st = check_head_layout(host ? W : step_hidden[k], ldh_elems, W, ldw_elems, H);
        if (st != CD_OK) return st;
        if (!step_hidden[k]) return fail(CD_ERR_ARG, "step_hidden[%d] is NULL", k);
    }
    RangeGuard range("cd_head_decode_loop");
    DeviceGuard guard(d->device);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const Settings cfg = settings_of(d);
    Scratch* s = nullptr;
    st = get_scratch(d, stream, B, &s);
    if (st != CD_OK) return st;
    int* d_tokens = tokens_out;
    int* d_len = len_out;
    int* d_fs = final_state_out;
    float* d_slp = sum_logprob_out;
    uint8_t* d_done = done_out;
    const size_t step_bytes = (size_t)B * (size_t)ldh_elems * 2;
    const size_t n_tok = (size_t)B * (size_t)(max_steps > 0 ? max_steps : 1);
    if (host) {
        // two staging buffers: the H2D copy of step k + 1 overlaps the kernels of step k
        const size_t out_bytes = sizeof(int) * (n_tok + 3 * (size_t)B) + (size_t)B + 64;
        st = get_host_loop_scratch(s, step_bytes, step_bytes, out_bytes, stream);
        if (st != CD_OK) return st;
        d_tokens = s->out_i32;
        d_len = d_tokens + n_tok;
        d_fs = d_len + B;
        d_slp = reinterpret_cast<float*>(d_fs + B);
        d_done = reinterpret_cast<uint8_t*>(d_slp + B);
    }
    const LimitArgs lim = resolve_limit(cfg);
    st = launch_loop_init(d, s, B, max_steps, d_tokens, d_len, d_fs, d_slp, d_done, stream, lim);
    if (st != CD_OK) return st;
    if (!d->start_accepting && max_steps > 0) {
        st = get_head_scratch(s, B, H, stream);
        if (st != CD_OK) return st;
        if (host) {
            CU(cudaEventRecord(s->ev_consumed[0], stream));
            CU(cudaEventRecord(s->ev_consumed[1], stream));
            CU(cudaStreamWaitEvent(s->copy_stream, s->ev_consumed[0], 0));
            CU(cudaMemcpyAsync(s->stage[0], step_hidden[0], step_bytes, cudaMemcpyHostToDevice, s->copy_stream));
            CU(cudaEventRecord(s->ev_copied[0], s->copy_stream));
        }
        for (int k = 0; k < max_steps; ++k) {
            const int cur = k & 1, nxt = cur ^ 1;
            const void* hid = step_hidden[k];
            if (host) {
                if (k + 1 < max_steps) {
                    CU(cudaStreamWaitEvent(s->copy_stream, s->ev_consumed[nxt], 0));
                    CU(cudaMemcpyAsync(s->stage[nxt], step_hidden[k + 1], step_bytes, cudaMemcpyHostToDevice,
                                       s->copy_stream));
                    CU(cudaEventRecord(s->ev_copied[nxt], s->copy_stream));
                }
                CU(cudaStreamWaitEvent(stream, s->ev_copied[cur], 0));
                hid = s->stage[cur];
            }
            LoopExtras x;
            x.tokens = d_tokens;
            x.len = d_len;
            x.final_state = d_fs;
            x.sum_logprob = d_slp;
            x.done = d_done;
            x.step = k;
            x.max_steps = max_steps;
            x.row_ids_out = s->b.row_ids[nxt];
            x.state_out = s->b.state[nxt];
            x.n_out = s->b.n_active + nxt;
            if (lim.sat_ctr) {
                x.satisfying = static_cast<const uint8_t*>(d->d_satisfying);
                x.sat_ctr = lim.sat_ctr;
                x.limit = lim.limit;
            }
            RangeGuard step_range("cd decoding step (LM head)");
            st = launch_head(d, cfg, s, hid, ldh_elems, W, ldw_elems, H, s->b.row_ids[cur], s->b.state[cur], B,
                             s->b.n_active + cur, s->b.token, s->b.logprob, nullptr, s->b.done, stream, &x);
            if (st != CD_OK) return st;
            if (host) CU(cudaEventRecord(s->ev_consumed[cur], stream));
        }
        if (host) CU(cudaStreamSynchronize(s->copy_stream));
    }
    if (host) {
        if (max_steps > 0)
            CU(cudaMemcpyAsync(tokens_out, d_tokens, sizeof(int) * (size_t)B * max_steps, cudaMemcpyDeviceToHost, stream));
        CU(cudaMemcpyAsync(len_out, d_len, sizeof(int) * (size_t)B, cudaMemcpyDeviceToHost, stream));
        CU(cudaMemcpyAsync(final_state_out, d_fs, sizeof(int) * (size_t)B, cudaMemcpyDeviceToHost, stream));
        CU(cudaMemcpyAsync(sum_logprob_out, d_slp, sizeof(float) * (size_t)B, cudaMemcpyDeviceToHost, stream));
        CU(cudaMemcpyAsync(done_out, d_done, (size_t)B, cudaMemcpyDeviceToHost, stream));
    }
    return finish_loop(s, stream, false);
}

cd_status cd_head_decode_loop(const cd_dfa_t* d, const void* const* step_hidden, int64_t ldh_elems, const void* W,
                              int64_t ldw_elems, int32_t H, int32_t B, int32_t max_steps, int32_t* tokens_out,
                              int32_t* len_out, int32_t* final_state_out, float* sum_logprob_out, uint8_t* done_out,
                              void* cuda_stream) {
    return head_loop_impl(d, step_hidden, false, ldh_elems, W, ldw_elems, H, B, max_steps, tokens_out, len_out,
                          final_state_out, sum_logprob_out, done_out, cuda_stream);
}

cd_status cd_head_decode_loop_host(const cd_dfa_t* d, const void* const* step_hidden_host, int64_t ldh_elems,
                                   const void* W, int64_t ldw_elems, int32_t H, int32_t B, int32_t max_steps,
                                   int32_t* tokens_out, int32_t* len_out, int32_t* final_state_out,
                                   float* sum_logprob_out, uint8_t* done_out, void* cuda_stream) {
    return head_loop_impl(d, step_hidden_host, true, ldh_elems, W, ldw_elems, H, B, max_steps, tokens_out, len_out,
                          final_state_out, sum_logprob_out, done_out, cuda_stream);
}

}  // extern "C"

// =============================================================================== dedup / join / cascade
namespace {

int grid_for(long long n, int threads) {
    long long b = (n + threads - 1) / threads;
    if (b < 1) b = 1;
    if (b > 148 * 16) b = 148 * 16;
    return (int)b;
}

}  // namespace

extern "C" {

cd_status cd_probe_read(const void* buf, int64_t bytes, int32_t iters, float* ms_out, void* cuda_stream) {
    if (!buf || bytes < 8192 || iters < 1 || !ms_out) return fail(CD_ERR_ARG, "bad argument");
    if ((reinterpret_cast<uintptr_t>(buf) & 15) != 0) return fail(CD_ERR_ARG, "buffer is not 16-byte aligned");
    int dev = 0;
    cd_status st = device_of(buf, &dev);
    if (st != CD_OK) return st;
    DeviceGuard guard(dev);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    constexpr int W = 12, S = 2, T = 8192;
    auto kern = cd::read_probe_kernel<W, S, T>;
    const size_t smem = (size_t)W * S * T;
    CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, dev));
    const unsigned long long ntiles = (unsigned long long)bytes / T;
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0));
    CU(cudaEventCreate(&e1));
    for (int i = 0; i < 2; ++i) kern<<<prop.multiProcessorCount, W * 32, smem, stream>>>(static_cast<const unsigned char*>(buf), ntiles, nullptr);
    CU(cudaEventRecord(e0, stream));
    for (int i = 0; i < iters; ++i) kern<<<prop.multiProcessorCount, W * 32, smem, stream>>>(static_cast<const unsigned char*>(buf), ntiles, nullptr);
    CU(cudaEventRecord(e1, stream));
    CU(cudaEventSynchronize(e1));
    CU(cudaGetLastError());
    float ms = 0.0f;
    CU(cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    g_launches.fetch_add(iters + 2, std::memory_order_relaxed);
    *ms_out = ms / iters;
    return CD_OK;
}

cd_status cd_dedup(const int64_t* keys, int32_t N, int32_t* rep_out, int32_t* distinct_rows_out,
                   int32_t* n_distinct_out, void* cuda_stream) {
    if (N < 0) return fail(CD_ERR_ARG, "N < 0");
    if (!n_distinct_out) return fail(CD_ERR_ARG, "n_distinct_out is NULL");
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    int dev = 0;
    cd_status st = device_of(n_distinct_out, &dev);
    if (st != CD_OK) return st;
    DeviceGuard guard(dev);
    keep_pool_memory(dev);
    if (N == 0) {
        CU(cudaMemsetAsync(n_distinct_out, 0, sizeof(int), stream));
        return CD_OK;
    }
    if (!keys || !rep_out || !distinct_rows_out) return fail(CD_ERR_ARG, "NULL pointer");
    if (N > (1 << 30)) return fail(CD_ERR_ARG, "N (%d) exceeds 2^30 rows per call", N);  // table of 2N..4N 32-bit slots
    uint32_t cap = 1024;
    while (cap < 2ull * (uint32_t)N) cap <<= 1;
    // stream-ordered scratch: table keys [cap + 1], table min rows [cap + 1], first [N], rank [N], flags [N]
    const size_t off_min = sizeof(unsigned long long) * ((size_t)cap + 1);
    const size_t off_first = off_min + sizeof(int) * ((size_t)cap + 1 + 3) / 16 * 16 + 16;
    const size_t off_rank = off_first + sizeof(int) * (size_t)N;
    const size_t off_flag = off_rank + sizeof(int) * (size_t)N;
    const size_t total = off_flag + (size_t)N + 16;
    unsigned char* buf = nullptr;
    CU(cudaMallocAsync(reinterpret_cast<void**>(&buf), total, stream));
    unsigned long long* tkey = reinterpret_cast<unsigned long long*>(buf);
    int* tmin = reinterpret_cast<int*>(buf + off_min);
    int* first = reinterpret_cast<int*>(buf + off_first);
    int* rank = reinterpret_cast<int*>(buf + off_rank);
    uint8_t* flag = buf + off_flag;
    // min rows start at 0x7F7F7F7F (>= any row id); free slots hold DEDUP_EMPTY
    cudaError_t e = cudaMemsetAsync(tmin, 0x7F, sizeof(int) * ((size_t)cap + 1), stream);
    if (e == cudaSuccess) {
        cd::dedup_clear_kernel<<<grid_for((long long)cap + 1, 256), 256, 0, stream>>>(tkey, (long long)cap + 1);
        cd::dedup_insert_kernel<<<grid_for(N, 256), 256, 0, stream>>>(reinterpret_cast<const long long*>(keys), N, tkey, tmin, cap);
        cd::dedup_first_kernel<<<grid_for(N, 256), 256, 0, stream>>>(reinterpret_cast<const long long*>(keys), N, tkey, tmin,
                                                                   cap, first, flag);
        e = cudaGetLastError();
    }
    // stable ranking of the first occurrences: the compaction of a6 over the "not first" flags (ids = row numbers),
    // with the output position of every kept row recorded
    st = (e == cudaSuccess) ? launch_compact(flag, nullptr, nullptr, N, distinct_rows_out, nullptr, n_distinct_out, rank, stream)
                            : fail(CD_ERR_CUDA, "dedup launch: %s", cudaGetErrorString(e));
    if (st == CD_OK) {
        cd::dedup_rep_kernel<<<grid_for(N, 256), 256, 0, stream>>>(first, rank, N, rep_out);
        e = cudaGetLastError();
        if (e != cudaSuccess) st = fail(CD_ERR_CUDA, "dedup launch: %s", cudaGetErrorString(e));
    }
    cudaFreeAsync(buf, stream);  // on every path
    if (st == CD_OK) g_launches.fetch_add(4, std::memory_order_relaxed);
    return st;
}

cd_status cd_join_results(const int32_t* rep, int32_t N, int32_t max_steps, const int32_t* tokens_d, const int32_t* len_d,
                          const int32_t* final_state_d, const float* sum_logprob_d, const uint8_t* done_d,
                          int32_t* tokens_out, int32_t* len_out, int32_t* final_state_out, float* sum_logprob_out,
                          uint8_t* done_out, void* cuda_stream) {
    if (N < 0 || max_steps < 0) return fail(CD_ERR_ARG, "N / max_steps < 0");
    if (N == 0) return CD_OK;
    if (!rep) return fail(CD_ERR_ARG, "rep is NULL");
    if ((tokens_out && !tokens_d) || (len_out && !len_d) || (final_state_out && !final_state_d) ||
        (sum_logprob_out && !sum_logprob_d) || (done_out && !done_d))
        return fail(CD_ERR_ARG, "an output is requested without its source");
    int dev = 0;
    cd_status st = device_of(rep, &dev);
    if (st != CD_OK) return st;
    DeviceGuard guard(dev);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    int vec_lanes = 0;  // lanes per token row on the 16-byte path (cd_dedup.cuh), 0 = element-wise copy
    if (tokens_out && max_steps > 0 && max_steps % 4 == 0 && ((reinterpret_cast<uintptr_t>(tokens_out) | reinterpret_cast<uintptr_t>(tokens_d)) & 15) == 0) {
        vec_lanes = 1;
        while (vec_lanes < 32 && vec_lanes < max_steps / 4) vec_lanes <<= 1;
    }
    const long long threads = vec_lanes ? (long long)N * vec_lanes : (long long)N * (max_steps > 0 ? max_steps : 1);
    cd::join_kernel<<<grid_for(threads, 256), 256, 0, stream>>>(
        rep, N, max_steps, tokens_d, len_d, final_state_d, sum_logprob_d, done_d, max_steps > 0 ? tokens_out : nullptr,
        len_out, final_state_out, sum_logprob_out, done_out, vec_lanes);
    CU(cudaGetLastError());
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return CD_OK;
}

cd_status cd_filter_rows(const cd_dfa_t* d, const int32_t* final_state, const uint8_t* done, const int32_t* row_ids_in,
                         int32_t N, int32_t* row_ids_out, int32_t* n_out, void* cuda_stream) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (!settings_of(d).has_satisfying) return fail(CD_ERR_ARG, "cd_set_satisfying has not been called on this automaton");
    if (N < 0) return fail(CD_ERR_ARG, "N < 0");
    if (!n_out) return fail(CD_ERR_ARG, "n_out is NULL");
    DeviceGuard guard(d->device);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (N == 0) {
        CU(cudaMemsetAsync(n_out, 0, sizeof(int), stream));
        return CD_OK;
    }
    if (!final_state || !done || !row_ids_out) return fail(CD_ERR_ARG, "NULL pointer");
    keep_pool_memory(d->device);
    uint8_t* drop = nullptr;
    CU(cudaMallocAsync(reinterpret_cast<void**>(&drop), (size_t)N + 16, stream));
    cd::filter_flag_kernel<<<grid_for(N, 256), 256, 0, stream>>>(final_state, done, N,
                                                               static_cast<const uint8_t*>(d->d_satisfying), d->dev.S, drop);
    const cudaError_t e = cudaGetLastError();
    const cd_status st = (e == cudaSuccess) ? launch_compact(drop, row_ids_in, nullptr, N, row_ids_out, nullptr, n_out, nullptr, stream)
                                            : fail(CD_ERR_CUDA, "filter launch: %s", cudaGetErrorString(e));
    cudaFreeAsync(drop, stream);  // on every path
    if (st == CD_OK) g_launches.fetch_add(1, std::memory_order_relaxed);
    return st;
}

}  // extern "C"

// =============================================================================== callback loops
extern "C" {

cd_status cd_decode_loop_cb(const cd_dfa_t* d, cd_next_logits_fn next_logits, void* user, cd_dtype dtype, int32_t B,
                            int32_t max_steps, int32_t* tokens_out, int32_t* len_out, int32_t* final_state_out,
                            float* sum_logprob_out, uint8_t* done_out, void* cuda_stream) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (!next_logits) return fail(CD_ERR_ARG, "next_logits is NULL");
    if (B < 0 || max_steps < 0) return fail(CD_ERR_ARG, "B / max_steps < 0");
    cd_status st = check_dtype(dtype);
    if (st != CD_OK) return st;
    if (B == 0) return CD_OK;
    if (!len_out || !final_state_out || !sum_logprob_out || !done_out || (max_steps > 0 && !tokens_out))
        return fail(CD_ERR_ARG, "NULL output pointer");
    DeviceGuard guard(d->device);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    RangeGuard range("cd_decode_loop_cb");
    const Settings cfg = settings_of(d);
    Scratch* s = nullptr;
    st = get_scratch(d, stream, B, &s);
    if (st != CD_OK) return st;
    const LimitArgs lim = resolve_limit(cfg);
    st = launch_loop_init(d, s, B, max_steps, tokens_out, len_out, final_state_out, sum_logprob_out, done_out, stream,
                          lim);
    if (st != CD_OK) return st;
    if (!d->start_accepting)
        for (int k = 0; k < max_steps; ++k) {
            const int cur = k & 1;
            const void* logits = nullptr;
            int64_t ld = 0;
            int32_t by_slot = 0;
            const int rc = next_logits(user, k, s->b.row_ids[cur], s->b.n_active + cur, B, &logits, &ld, &by_slot);
            if (rc != 0) return fail(CD_ERR_ARG, "next_logits returned %d at step %d", rc, k);
            st = check_logits_layout(d, logits, dtype, ld);
            if (st != CD_OK) return st;
            st = enqueue_loop_step(d, cfg, s, logits, dtype, ld, B, k, max_steps, tokens_out, len_out, final_state_out,
                                   sum_logprob_out, done_out, stream, lim, by_slot ? 1 : 0);
            if (st != CD_OK) return st;
        }
    return finish_loop(s, stream, false);
}

cd_status cd_head_decode_loop_cb(const cd_dfa_t* d, cd_next_hidden_fn next_hidden, void* user, const void* W,
                                 int64_t ldw_elems, int32_t H, int32_t B, int32_t max_steps, int32_t* tokens_out,
                                 int32_t* len_out, int32_t* final_state_out, float* sum_logprob_out, uint8_t* done_out,
                                 void* cuda_stream) {
    if (!d) return fail(CD_ERR_ARG, "dfa is NULL");
    if (!next_hidden) return fail(CD_ERR_ARG, "next_hidden is NULL");
    if (B < 0 || max_steps < 0) return fail(CD_ERR_ARG, "B / max_steps < 0");
    if (B == 0) return CD_OK;
    if (!len_out || !final_state_out || !sum_logprob_out || !done_out || (max_steps > 0 && !tokens_out))
        return fail(CD_ERR_ARG, "NULL output pointer");
    DeviceGuard guard(d->device);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    RangeGuard range("cd_head_decode_loop_cb");
    const Settings cfg = settings_of(d);
    Scratch* s = nullptr;
    cd_status st = get_scratch(d, stream, B, &s);
    if (st != CD_OK) return st;
    const LimitArgs lim = resolve_limit(cfg);
    st = launch_loop_init(d, s, B, max_steps, tokens_out, len_out, final_state_out, sum_logprob_out, done_out, stream,
                          lim);
    if (st != CD_OK) return st;
    if (!d->start_accepting && max_steps > 0) {
        st = get_head_scratch(s, B, H, stream);
        if (st != CD_OK) return st;
        for (int k = 0; k < max_steps; ++k) {
            const int cur = k & 1, nxt = cur ^ 1;
            const void* hidden = nullptr;
            int64_t ldh = 0;
            int32_t by_slot = 0;
            const int rc = next_hidden(user, k, s->b.row_ids[cur], s->b.n_active + cur, B, &hidden, &ldh, &by_slot);
            if (rc != 0) return fail(CD_ERR_ARG, "next_hidden returned %d at step %d", rc, k);
            st = check_head_layout(hidden, ldh, W, ldw_elems, H);
            if (st != CD_OK) return st;
            LoopExtras x;
            x.tokens = tokens_out;
            x.len = len_out;
            x.final_state = final_state_out;
            x.sum_logprob = sum_logprob_out;
            x.done = done_out;
            x.step = k;
            x.max_steps = max_steps;
            x.row_ids_out = s->b.row_ids[nxt];
            x.state_out = s->b.state[nxt];
            x.n_out = s->b.n_active + nxt;
            x.logits_by_slot = by_slot ? 1 : 0;
            if (lim.sat_ctr) {
                x.satisfying = static_cast<const uint8_t*>(d->d_satisfying);
                x.sat_ctr = lim.sat_ctr;
                x.limit = lim.limit;
            }
            RangeGuard step_range("cd decoding step (LM head)");
            st = launch_head(d, cfg, s, hidden, ldh, W, ldw_elems, H, s->b.row_ids[cur], s->b.state[cur], B,
                             s->b.n_active + cur, s->b.token, s->b.logprob, nullptr, s->b.done, stream, &x);
            if (st != CD_OK) return st;
        }
    }
    return finish_loop(s, stream, false);
}

}  // extern "C"

// =============================================================================== typed-output sugar
extern "C" {

cd_status cd_build_list(int32_t V, int32_t K, const int64_t* label_ptr, const int32_t* label_tok, const int32_t* open,
                        int32_t n_open, const int32_t* sep, int32_t n_sep, const int32_t* close, int32_t n_close,
                        int32_t min_items, int32_t max_items, int32_t eos, int32_t* S_out, int64_t* nnz_out,
                        int64_t* row_ptr_out, int32_t* tok_out, int32_t* next_out, uint8_t* accepting_out) {
    try {
        if (!label_ptr || !S_out || !nnz_out) return fail(CD_ERR_ARG, "NULL argument");
        if (K >= 1 && label_ptr[K] > 0 && !label_tok) return fail(CD_ERR_ARG, "label_tok is NULL");
        if ((n_open > 0 && !open) || (n_sep > 0 && !sep) || (n_close > 0 && !close)) return fail(CD_ERR_ARG, "NULL token list");
        cdt::HostCsr c;
        const std::string err = cdt::build_list(V, K, label_ptr, label_tok, open, n_open, sep, n_sep, close, n_close,
                                                min_items, max_items, eos, &c);
        if (!err.empty()) return fail(CD_ERR_AUTOMATON, "%s", err.c_str());
        return copy_csr_out(c, S_out, nnz_out, row_ptr_out, tok_out, next_out, accepting_out);
    } catch (const std::bad_alloc&) {
        return fail(CD_ERR_OOM, "host allocation failed");
    } catch (...) {
        return fail(CD_ERR_INTERNAL, "unexpected exception");
    }
}

cd_status cd_compile_list(int32_t V, int32_t K, const int64_t* label_ptr, const int32_t* label_tok, const int32_t* open,
                          int32_t n_open, const int32_t* sep, int32_t n_sep, const int32_t* close, int32_t n_close,
                          int32_t min_items, int32_t max_items, int32_t eos, int device, cd_dfa_t** out) {
    try {
        if (!label_ptr || !out) return fail(CD_ERR_ARG, "NULL argument");
        if ((n_open > 0 && !open) || (n_sep > 0 && !sep) || (n_close > 0 && !close)) return fail(CD_ERR_ARG, "NULL token list");
        cdt::HostCsr c;
        const std::string err = cdt::build_list(V, K, label_ptr, label_tok, open, n_open, sep, n_sep, close, n_close,
                                                min_items, max_items, eos, &c);
        if (!err.empty()) return fail(CD_ERR_AUTOMATON, "%s", err.c_str());
        return compile_csr(V, c, device, out);
    } catch (const std::bad_alloc&) {
        return fail(CD_ERR_OOM, "host allocation failed");
    } catch (...) {
        return fail(CD_ERR_INTERNAL, "unexpected exception");
    }
}

}  // extern "C"
