// cd_common.cuh -- device-side structs and sm_100a PTX helpers shared by the kernels.
// Part of the product path (never included by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cd {

constexpr unsigned FULL = 0xFFFFFFFFu;
constexpr int DT_F32 = 0;
constexpr int DT_BF16 = 1;

// Device image of a compiled automaton.
struct DfaDev {
    int V;                     // vocabulary size
    int S;                     // number of states
    int W;                     // ceil(V / 32) mask words that carry bits
    int Wpad;                  // mask row stride in words, multiple of 4 (16 B rows), pad = 0
    const uint32_t* mask;      // [S][Wpad], LSB-first: token t <-> bit (t & 31) of word (t >> 5)
    const long long* row_ptr;  // [S + 1]
    const int* tok;            // [nnz] strictly increasing inside a state
    const int* next;           // [nnz] next state | (accepting[next state] << 31)
    const uint8_t* accepting;  // [S]
    const int* rank1k;         // [S][nblk] number of allowed tokens of the state below token 1024 * b
    int nblk;                  // ceil(V / 1024)
};

// ---------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}

__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void fence_proxy_async_smem() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
}

__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t"
        "}" ::"r"(bar),
        "r"(parity)
        : "memory");
}

// Programmatic dependent launch (sm_90+): see step_kernel.
__device__ __forceinline__ void pdl_launch_dependents() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
__device__ __forceinline__ void pdl_wait() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}

__device__ __forceinline__ uint64_t l2_policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}

// Device-scope acquire-release add: earlier writes of this thread are visible to whoever
// observes the new counter value; later reads of this thread see what earlier arrivers wrote.
__device__ __forceinline__ int atom_add_acq_rel_gpu(int* p, int v) {
    int old;
    asm volatile("atom.add.acq_rel.gpu.global.s32 %0, [%1], %2;" : "=r"(old) : "l"(p), "r"(v) : "memory");
    return old;
}

// 1-D bulk async copy global -> shared (TMA engine, SASS UBLKCP), completion on an mbarrier.
// dst, src 16-byte aligned; bytes a positive multiple of 16.
__device__ __forceinline__ void bulk_g2s_hint(uint32_t dst, const void* src, uint32_t bytes,
                                              uint32_t bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint "
        "[%0], [%1], %2, [%3], %4;" ::"r"(dst),
        "l"(src), "r"(bytes), "r"(bar), "l"(policy)
        : "memory");
}

__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
        "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}

// ---------------------------------------------------------------- online softmax pieces
// (m, s, idx): running masked maximum, sum of exp(x - m) over the allowed elements seen so
// far, lowest token id attaining m.  Elements are presented in ascending token id per lane,
// so "replace on strictly greater" keeps the lowest id (north_star: ties -> lowest token id).
constexpr float LOG2E = 1.4426950408889634f;

__device__ __forceinline__ float ex2_ftz(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Branch-free.  x = -inf (a masked-out lane, or an allowed -inf / NaN logit) changes nothing.
// One MUFU per element: either the old sum or the new term is scaled by e = exp(-|x - m|).
__device__ __forceinline__ void online_update(float& m, float& s, int& idx, float x, int t) {
    const float lo = fminf(m, x), hi = fmaxf(m, x);
    float e = ex2_ftz((lo - hi) * LOG2E);
    e = (lo == -INFINITY) ? 0.0f : e;  // also covers m = x = -inf (lo - hi = NaN)
    const bool gt = x > m;
    s = gt ? fmaf(s, e, 1.0f) : s + e;
    idx = gt ? t : idx;
    m = hi;
}

// Merge two partial results; equal maxima keep the lower token id whatever the order.
__device__ __forceinline__ void online_combine(float& m, float& s, int& idx, float m2, float s2, int i2) {
    const bool take2 = (m2 > m) || (m2 == m && i2 < idx);
    const float mw = take2 ? m2 : m, ml = take2 ? m : m2;
    const float sw = take2 ? s2 : s, sl = take2 ? s : s2;
    const float f = (ml == -INFINITY) ? 0.0f : ex2_ftz((ml - mw) * LOG2E);
    s = fmaf(sl, f, sw);
    m = mw;
    idx = take2 ? i2 : idx;
}

__device__ __forceinline__ void warp_combine(float& m, float& s, int& idx) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float m2 = __shfl_xor_sync(FULL, m, o);
        const float s2 = __shfl_xor_sync(FULL, s, o);
        const int i2 = __shfl_xor_sync(FULL, idx, o);
        online_combine(m, s, idx, m2, s2, i2);
    }
}

// Warp combination through the redux unit: the maximum first (one REDUX on an order-preserving integer
// image of the float), every lane rescales its sum once, the sums are added in the xor-butterfly order
// (commutative pairs: every lane ends with the same bits), the token is the lowest id among the lanes that
// attain the maximum (one REDUX).  ~25 instructions and ~200 cycles instead of the 5 dependent online_combine
// rounds of warp_combine.  All lanes return the same (m, s, idx).
__device__ __forceinline__ int float_order_key(float x) {
    const int k = __float_as_int(x);
    return k >= 0 ? k : (k ^ 0x7FFFFFFF);
}
__device__ __forceinline__ float float_from_order_key(int k) {
    return __int_as_float(k >= 0 ? k : (k ^ 0x7FFFFFFF));
}
__device__ __forceinline__ void warp_combine_redux(float& m, float& s, int& idx) {
    const float M = float_from_order_key(__reduce_max_sync(FULL, float_order_key(m)));
    const float f = (m == -INFINITY) ? 0.0f : ex2_ftz((m - M) * LOG2E);
    float t = s * f;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(FULL, t, o);
    const unsigned cand = (m == M) ? (unsigned)idx : 0xFFFFFFFFu;
    idx = (int)__reduce_min_sync(FULL, cand);
    m = M;
    s = t;
}
// the same for the sampling key: the largest perturbed key, ties to the lowest id
__device__ __forceinline__ void warp_argmax_redux(float& kb, int& kidx) {
    const float K = float_from_order_key(__reduce_max_sync(FULL, float_order_key(kb)));
    const unsigned cand = (kb == K) ? (unsigned)kidx : 0xFFFFFFFFu;
    kidx = (int)__reduce_min_sync(FULL, cand);
    kb = K;
}

// ---------------------------------------------------------------- sampling
// Gumbel-max over the allowed set with a counter-based generator: the noise of (row, step, token)
// is a pure function of the seed, so results do not depend on launch shape, compaction or the
// order rows are processed in.  Every operation below is an IEEE-754 correctly rounded fp32
// operation (explicit _rn intrinsics: never contracted or reordered) or integer arithmetic, so the
// CPU oracle, which restates the same definition in C, decides the argmax on identical bits.
__device__ __forceinline__ uint32_t fmix32(uint32_t h) {
    h ^= h >> 16;
    h *= 0x85EBCA6Bu;
    h ^= h >> 13;
    h *= 0xC2B2AE35u;
    h ^= h >> 16;
    return h;
}

// per (row, step) part of the counter hash
__device__ __forceinline__ uint32_t rng_row_key(uint32_t seed_lo, uint32_t seed_hi, uint32_t row, uint32_t step) {
    uint32_t h = fmix32(seed_lo ^ (row * 0x9E3779B1u));
    return fmix32(h ^ (step * 0x85EBCA77u) ^ seed_hi);
}

// natural logarithm of a positive normal fp32 from +, *, /, fma only:
// x = m * 2^e with m in [sqrt(1/2), sqrt(2)); ln m = 2 atanh(s), s = (m - 1) / (m + 1), odd series to s^9
__device__ __forceinline__ float det_logf(float x) {
    const int ix = __float_as_int(x);
    const int e = (ix - 0x3F3504F3) >> 23;
    const float m = __int_as_float(ix - (e << 23));
    const float f = __fadd_rn(m, -1.0f);
    const float sden = __fadd_rn(2.0f, f);
    const float sq = __fdiv_rn(f, sden);
    const float z = __fmul_rn(sq, sq);
    float p = __fmaf_rn(z, 0.111111111f, 0.142857143f);
    p = __fmaf_rn(z, p, 0.2f);
    p = __fmaf_rn(z, p, 0.333333333f);
    p = __fmaf_rn(z, p, 1.0f);
    const float r = __fmul_rn(__fmul_rn(2.0f, sq), p);
    return __fmaf_rn((float)e, 0.693147181f, r);
}

// Gumbel(0,1) noise of token `tok`: u = (2b + 1) / 2^24 with b = top 23 hash bits (exact in fp32,
// inside (0,1)), g = -ln(-ln u)
__device__ __forceinline__ float gumbel_noise(uint32_t row_key, uint32_t tok) {
    const uint32_t h = fmix32(fmix32(row_key ^ (tok * 0xC2B2AE3Du)) + 0x27D4EB2Fu);
    const float u = __fmul_rn((float)(2u * (h >> 9) + 1u), 5.9604644775390625e-8f);  // * 2^-24, exact
    const float l1 = -det_logf(u);  // in [2^-24.x, 16.7]
    return -det_logf(l1);
}

// Online update of the sampling state: (m, s) over y = x * inv_tau as in online_update, plus the
// running best perturbed key and its token (ascending ids per lane: strictly greater replaces).
__device__ __forceinline__ void online_update_sample(float& m, float& s, float& kb, int& kidx, float x, int t, int pos,
                                                     float inv_tau, uint32_t row_key) {
    const float y = fmaxf(__fmul_rn(x, inv_tau), -INFINITY);
    const float lo = fminf(m, y), hi = fmaxf(m, y);
    float e = ex2_ftz((lo - hi) * LOG2E);
    e = (lo == -INFINITY) ? 0.0f : e;
    s = (y > m) ? fmaf(s, e, 1.0f) : s + e;
    m = hi;
    const float key = __fadd_rn(y, gumbel_noise(row_key, (uint32_t)t));
    const bool gt = key > kb;
    kb = gt ? key : kb;
    kidx = gt ? pos : kidx;
}

__device__ __forceinline__ void sample_combine(float& kb, int& kidx, float k2, int i2) {
    const bool take2 = (k2 > kb) || (k2 == kb && i2 < kidx);
    kb = take2 ? k2 : kb;
    kidx = take2 ? i2 : kidx;
}

// ---------------------------------------------------------------- CSR transition lookup
// Warp-cooperative 128-ary search of `token` in the sorted CSR row tok[lo, hi): every round each
// lane probes 4 of 128 split points (independent loads), so a row of <= 4096 entries needs one
// round plus the final 32-wide compare, a 5,243-entry row (configs[3]) two: 2-3 dependent
// memory latencies instead of 13 for a binary search.  Returns the position or -1; all lanes
// return the same value.
__device__ __forceinline__ long long warp_csr_find(const int* __restrict__ tok, long long lo,
                                                   long long hi, int token, int lane) {
    while (hi - lo > 32) {
        const long long step = (hi - lo + 127) >> 7;
        int v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const long long q = lo + (long long)(lane * 4 + k) * step;
            v[k] = (q < hi) ? __ldg(tok + q) : 0x7FFFFFFF;
        }
        int c = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) c += __popc(__ballot_sync(FULL, v[k] <= token));
        if (c == 0) return -1;  // token below the first entry
        lo = lo + (long long)(c - 1) * step;
        hi = (lo + step < hi) ? lo + step : hi;
    }
    const long long q = lo + lane;
    const bool eq = (q < hi) && (__ldg(tok + q) == token);
    const unsigned b = __ballot_sync(FULL, eq);
    return b ? lo + (__ffs(b) - 1) : -1;
}

// Relaxed device-scope 64-bit accesses for the tagged partial-result slots (cd_step.cuh).
__device__ __forceinline__ void st_relaxed_gpu_u64(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_relaxed_gpu_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ int ld_relaxed_gpu_s32(const int* p) {
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// ---------------------------------------------------------------- stable compaction
// Active-row compaction by one CTA: every thread takes 4 consecutive slots,
// keep flags are counted per thread, prefix-summed over the warp with shuffles, over the warps
// through shared memory, and the running base is carried across chunks of 4*blockDim slots.
// Output order = input order (stable).  Inputs are read with ld.cg: in the fused path they were
// written by other SMs during the same kernel.  blockDim.x must be a multiple of 32, <= 1024.
__device__ __forceinline__ void block_compact(const uint8_t* __restrict__ done, const int* __restrict__ row_ids_in,
                                              const int* __restrict__ state_in, int n, int* __restrict__ row_ids_out,
                                              int* __restrict__ state_out, int* __restrict__ n_active_out) {
    __shared__ int s_warp[32];
    __shared__ int s_total;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
    // vector loads need 4-byte aligned flags and 16-byte aligned id / state lists
    const bool vec_ok = ((reinterpret_cast<uintptr_t>(done) & 3) == 0) &&
                        (!row_ids_in || (reinterpret_cast<uintptr_t>(row_ids_in) & 15) == 0) &&
                        (!state_in || (reinterpret_cast<uintptr_t>(state_in) & 15) == 0);
    int base = 0;
    for (int c0 = 0; c0 < n; c0 += 4 * (int)blockDim.x) {
        const int i0 = c0 + 4 * tid;
        int rid[4], st[4];
        bool keep[4];
        if (vec_ok && i0 + 3 < n) {
            const uint32_t d4 = __ldcg(reinterpret_cast<const uint32_t*>(done + i0));
#pragma unroll
            for (int q = 0; q < 4; ++q) keep[q] = ((d4 >> (8 * q)) & 0xFFu) == 0u;
            if (row_ids_in) {
                const int4 r4 = __ldcg(reinterpret_cast<const int4*>(row_ids_in + i0));
                rid[0] = r4.x; rid[1] = r4.y; rid[2] = r4.z; rid[3] = r4.w;
            } else {
#pragma unroll
                for (int q = 0; q < 4; ++q) rid[q] = i0 + q;
            }
            if (state_in) {
                const int4 s4 = __ldcg(reinterpret_cast<const int4*>(state_in + i0));
                st[0] = s4.x; st[1] = s4.y; st[2] = s4.z; st[3] = s4.w;
            }
        } else {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int i = i0 + q;
                keep[q] = (i < n) && (__ldcg(done + i) == 0);
                rid[q] = (i < n && row_ids_in) ? __ldcg(row_ids_in + i) : i;
                st[q] = (i < n && state_in) ? __ldcg(state_in + i) : 0;
            }
        }
        const int cnt = (int)keep[0] + (int)keep[1] + (int)keep[2] + (int)keep[3];
        int inc = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int u = __shfl_up_sync(FULL, inc, o);
            if (lane >= o) inc += u;
        }
        if (lane == 31) s_warp[warp] = inc;
        __syncthreads();
        if (warp == 0) {
            const int v = (lane < nwarps) ? s_warp[lane] : 0;
            int w = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int u = __shfl_up_sync(FULL, w, o);
                if (lane >= o) w += u;
            }
            s_warp[lane] = w - v;  // exclusive offset of each warp
            if (lane == 31) s_total = w;
        }
        __syncthreads();
        int pos = base + s_warp[warp] + inc - cnt;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (keep[q]) {
                row_ids_out[pos] = rid[q];
                if (state_in) state_out[pos] = st[q];
                ++pos;
            }
        }
        base += s_total;
        __syncthreads();
    }
    if (tid == 0) *n_active_out = base;
}

}  // namespace cd
