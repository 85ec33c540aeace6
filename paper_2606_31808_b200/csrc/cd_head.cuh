// cd_head.cuh -- the constrained step fused with the LM head (include/cd.h
// cd_head_step).  logits x_i[t] = <hidden_i, W[t]> are never written to HBM:
//
//   head_prepare_kernel  classifies the active slots by the density of their automaton state
//                        (accepting / gathered / dense) and builds the two work lists;
//   head_gather_kernel   low-density states (tries, option sets) and, in a late step of an early-exit loop,
//                        every row (automatic policy): work item = (row, piece of >= 128 transitions of its
//                        CSR token list), one CTA each; forms exactly the allowed logits as gathered dot
//                        products (W rows fetched in bursts) -- a one-piece row is finished by its CTA;
//   head_gather_finish_kernel  merges the pieces of the longer rows (masked logsumexp/argmax, transition);
//   head_pack_kernel     copies the hidden rows of the dense slots into a contiguous A operand;
//   head_dense_kernel    the dense contraction on the 5th-gen tensor cores for up to 128 dense rows:
//                        persistent, warp-specialised (TMA producer / tcgen05.mma issuer / 4 epilogue warps),
//                        128x256 fp32 accumulators double-buffered in TMEM, operands staged by
//                        TMA into 128B-swizzled shared memory.  The epilogue reads the
//                        accumulator rows with tcgen05.ld and applies the allowed-token bitmask
//                        of each row's own state to an online (max, sum-exp, argmax) -- one
//                        partial result per (row, range of vocabulary tiles);
//   head_dense2_kernel   the same on CTA pairs (clusters of 2, tcgen05.mma.cta_group::2, UMMA 256x256x16) for
//                        more than 128 dense rows: each CTA loads its 128 rows of A and half of the W tile;
//   head_finish_kernel   merges the partials of a dense row in a fixed order and does the CSR
//                        transition + accept test.
#pragma once
#include <cuda.h>

#include "cd_common.cuh"
#include "cd_step.cuh"

namespace cd {

constexpr int HD_BM = 128;   // rows per tile (UMMA M)
constexpr int HD_BN = 256;   // vocabulary entries per tile (UMMA N)
constexpr int HD_BK = 64;    // K per pipeline stage: 64 bf16 = one 128-byte swizzle row
constexpr int HD_UK = 16;    // K per tcgen05.mma (kind::f16)
constexpr int HD_STAGES = 4;
constexpr int HD_A_BYTES = HD_BM * HD_BK * 2;  // 16 KiB
constexpr int HD_B_BYTES = HD_BN * HD_BK * 2;  // 32 KiB
constexpr int HD_STAGE_BYTES = HD_A_BYTES + HD_B_BYTES;
constexpr int HD_SMEM_BYTES = HD_STAGES * HD_STAGE_BYTES + 1024;  // + slack to align to 1024 B
constexpr int HD_THREADS = 192;  // warp 0 TMA, warp 1 MMA + TMEM alloc, warps 2-5 epilogue
constexpr int HD_TMEM_COLS = 512;
constexpr int HD_UNITS_TARGET = 148 * 8;

constexpr int HG_WARPS = 8;      // gather kernel: warps per CTA
constexpr int HG_PIECE = 128;    // a gathered row is cut into pieces of >= this many transitions, one CTA each ...
constexpr int HG_MAX_PIECES = 64;  // ... at most this many per row
constexpr float HG_AUTO_FRAC = 0.8f;  // automatic policy: gather EVERY row while the W rows they touch are < 0.8 V (measured break-even on c3: ~0.9 V)

// canonical pieces of a gathered row of `deg` transitions (a function of deg only: results do not depend on the batch)
__host__ __device__ inline int hg_piece(int deg) {
    int p = (deg + HG_MAX_PIECES - 1) / HG_MAX_PIECES;
    p = (p + 7) & ~7;
    return p < HG_PIECE ? HG_PIECE : p;
}
__host__ __device__ inline int hg_pieces(int deg) {
    const int g = hg_piece(deg);
    const int n = (deg + g - 1) / g;
    return n < 1 ? 1 : n;
}

struct __align__(32) HeadPartial {
    float m, s;
    int idx;        // greedy: argmax token; sampling: sampled token
    float kb, yb;   // sampling: best perturbed key and the tempered logit of its token
    int pad[3];
};

// Sampling on the head path: as online_update_sample, and the tempered logit of the running winner is
// kept (the accumulator is gone once the tile is drained, so it cannot be re-read at finalisation).
__device__ __forceinline__ void head_update_sample(float& m, float& s, float& kb, int& kidx, float& yb, float x, int t,
                                                   int pos, float inv_tau, uint32_t row_key) {
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
    yb = gt ? y : yb;
}

__device__ __forceinline__ void head_sample_combine(float& kb, int& kidx, float& yb, float k2, int i2, float y2) {
    const bool take2 = (k2 > kb) || (k2 == kb && i2 < kidx);
    kb = take2 ? k2 : kb;
    kidx = take2 ? i2 : kidx;
    yb = take2 ? y2 : yb;
}

template <bool SAMPLE>
__device__ __forceinline__ void head_warp_combine(float& m, float& s, int& idx, float& kb, float& yb) {
    if constexpr (!SAMPLE) {
        warp_combine(m, s, idx);
    } else {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float m2 = __shfl_xor_sync(FULL, m, o), s2 = __shfl_xor_sync(FULL, s, o);
            const int i2 = __shfl_xor_sync(FULL, idx, o);
            const float k2 = __shfl_xor_sync(FULL, kb, o), y2 = __shfl_xor_sync(FULL, yb, o);
            int dummy = 0;
            online_combine(m, s, dummy, m2, s2, 0);
            head_sample_combine(kb, idx, yb, k2, i2, y2);
        }
    }
}

// Work decomposition of the dense contraction for n_dense rows: unit = (row tile, range of L
// consecutive vocabulary tiles); a row has NU partial results.  Unit u -> row tile u % num_m,
// range u / num_m, so that CTAs running at the same time share W tiles through L2.
struct HeadSched {
    int num_m, num_n, L, NU;
};
__host__ __device__ inline HeadSched head_sched(int n_dense, int V) {
    HeadSched h;
    h.num_m = (n_dense + HD_BM - 1) / HD_BM;
    h.num_n = (V + HD_BN - 1) / HD_BN;
    int nu0 = h.num_m > 0 ? (HD_UNITS_TARGET + h.num_m - 1) / h.num_m : 1;
    if (nu0 > h.num_n) nu0 = h.num_n;
    if (nu0 < 1) nu0 = 1;
    h.L = (h.num_n + nu0 - 1) / nu0;
    h.NU = (h.num_n + h.L - 1) / h.L;
    return h;
}
// upper bound of rows_pad * NU over n_dense <= n (capacity of the partial buffer)
__host__ inline long long head_partials_cap(int n) {
    const long long num_m = (n + HD_BM - 1) / HD_BM;
    return (long long)HD_BM * (HD_UNITS_TARGET + 2 * num_m + 2);
}

// ---- CTA-pair variant of the dense contraction (head_dense2_kernel, below)
constexpr int HD2_STAGES = 6;
constexpr int HD2_HALF_N = HD_BN / 2;                      // W rows each CTA loads
constexpr int HD2_B_BYTES = HD2_HALF_N * HD_BK * 2;        // 16 KiB
constexpr int HD2_STAGE_BYTES = HD_A_BYTES + HD2_B_BYTES;  // 32 KiB
constexpr int HD2_SMEM_BYTES = HD2_STAGES * HD2_STAGE_BYTES + 1024;
constexpr int HD2_UNITS_TARGET = 74 * 8;
constexpr int HD2_MIN_ROWS = HD_BM + 1;  // dense rows from which the pair kernel takes over

__host__ __device__ inline HeadSched head_sched2(int n_dense, int V) {  // num_m counts PAIRS of row tiles here
    HeadSched h;
    h.num_m = (n_dense + 2 * HD_BM - 1) / (2 * HD_BM);
    h.num_n = (V + HD_BN - 1) / HD_BN;
    int nu0 = h.num_m > 0 ? (HD2_UNITS_TARGET + h.num_m - 1) / h.num_m : 1;
    if (nu0 > h.num_n) nu0 = h.num_n;
    if (nu0 < 1) nu0 = 1;
    h.L = (h.num_n + nu0 - 1) / nu0;
    h.NU = (h.num_n + h.L - 1) / h.L;
    return h;
}
// partial results per dense row, whichever kernel runs the contraction
__host__ __device__ inline int head_row_partials(int n_dense, int V, int pairs) {
    return (pairs && n_dense >= HD2_MIN_ROWS) ? head_sched2(n_dense, V).NU : head_sched(n_dense, V).NU;
}

struct HeadArgs {
    StepArgs fin;  // dfa, outputs, sticky counters, optional loop history (see finalize_row);
                   // fin.state_new == fin.state: nothing reads state[] after head_prepare_kernel
    const uint16_t* hidden;  // [rows, ldh] bf16
    long long ldh;
    const uint16_t* W;  // [V, ldw] bf16
    long long ldw;
    int H;
    int gather_max;  // states with <= gather_max transitions are gathered
    int gather_auto; // automatic policy: when the rows above gather_max touch fewer than HG_AUTO_FRAC * V rows of W in
                     // total (a late step of an early-exit loop), they are gathered too instead of streaming all of W
    int gp_max;      // most pieces a gathered row of this call can have (bounds the item index)
    HeadPartial* gpartials;  // [rows][HG_MAX_PIECES] piece results of the gathered rows cut into several pieces
    int pairs;       // the CTA-pair kernel (head_dense2_kernel) is launched too and takes the calls with > 128 dense rows
    // scratch
    uint8_t* not_dense;   // [n]
    uint8_t* not_gather;  // [n]
    int* dense_slot;      // [n] slot of dense row d
    int* dense_state;     // [n]
    int* gather_slot;     // [n]
    int* gather_state;    // [n]
    int* hctr;            // [0] n_dense, [1] n_gather
    uint16_t* A;          // [rows_pad, ldA] packed hidden rows of the dense slots
    long long ldA;
    HeadPartial* partials;  // [rows_pad * NU]
};

// finalize_row's per-step view of a head step: next states go straight to state[] (== state_new)
__device__ __forceinline__ StepView head_view(const StepArgs& f) {
    StepView sv{};
    sv.state_next = f.state_new;
    sv.step = f.step;
    return sv;
}

// ---------------------------------------------------------------- sm_100a PTX: TMA, tcgen05
__device__ __forceinline__ void tma_prefetch_desc(const void* tmap) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(tmap)) : "memory");
}

// 2-D tiled TMA load global -> shared, completion (bytes) on an mbarrier.  c0 = inner coordinate.
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const void* tmap, int c0, int c1, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
        "l"(reinterpret_cast<uint64_t>(tmap)), "r"(c0), "r"(c1), "r"(bar)
        : "memory");
}

__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}

// tcgen05.commit: the mbarrier gets one arrival when every tcgen05.mma issued so far by this
// thread has completed (implies tcgen05.fence::before_thread_sync).
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

// D[tmem] (+)= A[smem] * B[smem]^T, bf16 x bf16 -> fp32, one thread issues for the CTA.
__device__ __forceinline__ void tc_mma_bf16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                            uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}

// Shared-memory matrix descriptor of a K-major tile whose rows are 128 bytes (64 bf16) in the
// 128-byte swizzle TMA writes: 8-row groups 1024 bytes apart (SBO), descriptor version 1
// (Blackwell), layout type 2 = SWIZZLE_128B.  The tile base is 1024-byte aligned; a K step of
// 16 elements inside the swizzle row advances the start address by 32 bytes.
__device__ __forceinline__ uint64_t umma_desc_k_sw128(uint32_t smem_addr) {
    return (uint64_t)((smem_addr >> 4) & 0x3FFFu) | (1ull << 16) | (64ull << 32) | (1ull << 46) | (2ull << 61);
}

// Instruction descriptor, kind::f16: D fp32 (bits 4-5 = 1), A and B bf16 (bits 7-9, 10-12 = 1),
// both K-major (bits 15, 16 = 0), N >> 3 at bits 17-22, M >> 4 at bits 24-28.
__host__ __device__ constexpr uint32_t umma_idesc_bf16(int M, int N) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

// 32 consecutive fp32 columns of this thread's TMEM lane (lane = quadrant base + laneid).
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// ---------------------------------------------------------------- prepare: classify + lists
// One CTA of 1024 threads.  A slot whose state already accepts (or is out of range) is finished
// here; the others go to the gather list (state has <= gather_max
// transitions) or to the dense list, both in slot order.
__global__ void __launch_bounds__(1024, 1) head_prepare_kernel(const HeadArgs a) {
    pdl_launch_dependents();  // launched with programmatic stream serialization: the next kernel may be scheduled,
    pdl_wait();               // and nothing of this one touches global memory before its predecessor has completed
    const StepArgs& f = a.fin;
    const int n = f.n_dev ? __ldcg(f.n_dev) : f.n;
    __shared__ unsigned long long s_big;  // transitions of the rows above gather_max, all together
    if (threadIdx.x == 0) s_big = 0ull;
    __syncthreads();
    unsigned long long big = 0ull;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const int st = f.state[i];
        const bool bad = (st < 0) || (st >= f.dfa.S);
        const bool acc = !bad && (__ldg(f.dfa.accepting + st) != 0);
        uint8_t nd = 1, ng = 1;
        if (bad || acc) {
            f.token_out[i] = -1;
            f.logprob_out[i] = 0.0f;
            if (f.lse_out) f.lse_out[i] = 0.0f;
            f.done_out[i] = 1;
            if (bad) atomicAdd(f.ctrs + 2, 1);
        } else {
            const int deg = (int)(__ldg(f.dfa.row_ptr + st + 1) - __ldg(f.dfa.row_ptr + st));
            if (deg <= a.gather_max) {
                ng = 0;
            } else {
                nd = 0;
                big += (unsigned long long)deg;
            }
        }
        a.not_dense[i] = nd;
        a.not_gather[i] = ng;
    }
    if (a.gather_auto) {  // one shared-memory atomic per warp (a 64-bit shared atomic is a CAS loop)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) big += __shfl_xor_sync(FULL, big, o);
        if ((threadIdx.x & 31) == 0 && big) atomicAdd(&s_big, big);
    }
    __syncthreads();
    // a dense step streams all V rows of W however few rows are left; gathering touches one W row per transition
    if (a.gather_auto && s_big > 0ull && (double)s_big < (double)HG_AUTO_FRAC * (double)f.dfa.V) {
        for (int i = threadIdx.x; i < n; i += blockDim.x)
            if (a.not_dense[i] == 0) {
                a.not_dense[i] = 1;
                a.not_gather[i] = 0;
            }
        __syncthreads();
    }
    block_compact(a.not_dense, nullptr, f.state, n, a.dense_slot, a.dense_state, a.hctr + 0);
    __syncthreads();
    block_compact(a.not_gather, nullptr, f.state, n, a.gather_slot, a.gather_state, a.hctr + 1);
}

// ---------------------------------------------------------------- pack: dense rows -> A
// One warp per dense row, 16-byte copies (H % 8 == 0, rows 16-byte aligned).
__global__ void head_pack_kernel(const HeadArgs a) {
    pdl_launch_dependents();  // launched with programmatic stream serialization: the next kernel may be scheduled,
    pdl_wait();               // and nothing of this one touches global memory before its predecessor has completed
    const int n_dense = __ldcg(a.hctr + 0);
    const int lane = threadIdx.x & 31;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int nwarps = (gridDim.x * blockDim.x) >> 5;
    const int nv = a.H >> 3;
    for (int d = warp; d < n_dense; d += nwarps) {
        const int slot = __ldcg(a.dense_slot + d);
        const long long r = (a.fin.row_map && !a.fin.logits_by_slot) ? (long long)__ldg(a.fin.row_map + slot) : (long long)slot;
        const uint4* src = reinterpret_cast<const uint4*>(a.hidden + r * a.ldh);
        uint4* dst = reinterpret_cast<uint4*>(a.A + (long long)d * a.ldA);
        for (int v = lane; v < nv; v += 32) dst[v] = __ldg(src + v);
    }
}

// ---------------------------------------------------------------- gather: low-density states
__device__ __forceinline__ float dot8(const uint4& w, const uint4& h, float acc) {
    const uint32_t wu[4] = {w.x, w.y, w.z, w.w}, hu[4] = {h.x, h.y, h.z, h.w};
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        acc = fmaf(__uint_as_float(wu[q] << 16), __uint_as_float(hu[q] << 16), acc);
        acc = fmaf(__uint_as_float(wu[q] & 0xFFFF0000u), __uint_as_float(hu[q] & 0xFFFF0000u), acc);
    }
    return acc;
}

// Work item = (gathered row g, piece p of its CSR token list), one CTA each (grid-stride): the hidden row is staged
// in shared memory, the warps split the piece into contiguous ranges, four dot products in flight per warp; the
// running argmax is the CSR position (ascending token id), so the transition needs no search.  A row of one piece
// (option sets, tries) is finished by its CTA; the piece results of a longer row go to gpartials and
// head_gather_finish_kernel merges them -- a late step with a handful of rows of thousands of transitions then
// spreads over the whole machine instead of keeping one SM per row busy.
// TWO: two W rows per warp at a time (16 loads per lane in flight, 112 registers: long rows cut into pieces); else one
// row at a time (8 loads, ~70 registers, one more CTA per SM: option sets, whose rows have a handful of transitions).
template <bool SAMPLE, bool TWO>
__global__ void __launch_bounds__(HG_WARPS * 32) head_gather_kernel(const HeadArgs a) {
    pdl_launch_dependents();  // launched with programmatic stream serialization: the next kernel may be scheduled,
    pdl_wait();               // and nothing of this one touches global memory before its predecessor has completed
    extern __shared__ __align__(16) unsigned char hg_smem[];
    uint4* hid = reinterpret_cast<uint4*>(hg_smem);
    __shared__ float s_m[HG_WARPS], s_s[HG_WARPS], s_k[HG_WARPS], s_y[HG_WARPS];
    __shared__ int s_i[HG_WARPS];
    const StepArgs& f = a.fin;
    const int n_gather = __ldcg(a.hctr + 1);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nv = a.H >> 3;
    const long long items = (long long)n_gather * a.gp_max;
    int staged = -1;  // gathered row whose hidden row is in shared memory
    for (long long it = blockIdx.x; it < items; it += gridDim.x) {
        const int g = (int)(it / a.gp_max), p = (int)(it - (long long)g * a.gp_max);
        const int slot = __ldcg(a.gather_slot + g);
        const int st = __ldcg(a.gather_state + g);
        const long long lo = __ldg(f.dfa.row_ptr + st);
        const int deg = (int)(__ldg(f.dfa.row_ptr + st + 1) - lo);
        const int np = hg_pieces(deg);
        if (p >= np) continue;  // (uniform over the CTA)
        const long long r = (f.row_map && !f.logits_by_slot) ? (long long)__ldg(f.row_map + slot) : (long long)slot;
        const uint4* src = reinterpret_cast<const uint4*>(a.hidden + r * a.ldh);
        __syncthreads();  // previous item's readers are done with hid / s_*
        if (staged != g) {
            for (int v = threadIdx.x; v < nv; v += blockDim.x) hid[v] = __ldg(src + v);
            staged = g;
        }
        __syncthreads();
        const int piece = hg_piece(deg);
        const int jlo = p * piece, jhi = min(deg, jlo + piece);
        const int j0 = jlo + (int)(((long long)(jhi - jlo) * warp) / HG_WARPS);
        const int j1 = jlo + (int)(((long long)(jhi - jlo) * (warp + 1)) / HG_WARPS);
        float m = -INFINITY, s = 0.0f, kb = -INFINITY, yb = -INFINITY;
        int idx = 0x7FFFFFFF;
        const uint32_t row_key =
            SAMPLE ? rng_row_key(f.seed_lo, f.seed_hi, (uint32_t)(f.row_map ? __ldg(f.row_map + slot) : slot),
                                 (uint32_t)(f.rng_step_base + f.step))
                   : 0u;
        // one or two W rows at a time, each read in passes of 8 x 512 contiguous bytes per warp with every load of the
        // pass in flight: a row is fetched in one or two bursts instead of being revisited chunk by chunk -- DRAM pages
        // are opened once
        constexpr int NR = TWO ? 2 : 1;
        for (int j = j0; j < j1; j += NR) {
            int tk[NR];
            const uint4* wr[NR];
#pragma unroll
            for (int q = 0; q < NR; ++q) {
                const int jq = (j + q < j1) ? j + q : j;
                tk[q] = __ldg(f.dfa.tok + lo + jq);
                wr[q] = reinterpret_cast<const uint4*>(a.W + (long long)tk[q] * a.ldw);
            }
            float acc[NR];
#pragma unroll
            for (int q = 0; q < NR; ++q) acc[q] = 0.0f;
            for (int v0 = lane; v0 < nv; v0 += 256) {
                uint4 x[NR][8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int v = v0 + 32 * u;
#pragma unroll
                    for (int q = 0; q < NR; ++q) x[q][u] = (v < nv) ? __ldg(wr[q] + v) : make_uint4(0, 0, 0, 0);
                }
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int v = v0 + 32 * u;
                    if (v < nv) {
                        const uint4 h = hid[v];
#pragma unroll
                        for (int q = 0; q < NR; ++q) acc[q] = dot8(x[q][u], h, acc[q]);
                    }
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
                for (int q = 0; q < NR; ++q) acc[q] += __shfl_xor_sync(FULL, acc[q], o);
            }
#pragma unroll
            for (int q = 0; q < NR; ++q)
                if (j + q < j1) {
                    if (SAMPLE)
                        head_update_sample(m, s, kb, idx, yb, fmaxf(acc[q], -INFINITY), tk[q], j + q, f.inv_tau, row_key);
                    else
                        online_update(m, s, idx, fmaxf(acc[q], -INFINITY), j + q);  // NaN -> -inf
                }
        }
        if (lane == 0) {
            s_m[warp] = m;
            s_s[warp] = s;
            s_i[warp] = idx;
            s_k[warp] = kb;
            s_y[warp] = yb;
        }
        __syncthreads();
        if (warp == 0) {
            float rm = (lane < HG_WARPS) ? s_m[lane] : -INFINITY;
            float rs = (lane < HG_WARPS) ? s_s[lane] : 0.0f;
            int ri = (lane < HG_WARPS) ? s_i[lane] : 0x7FFFFFFF;
            float rk = (lane < HG_WARPS) ? s_k[lane] : -INFINITY;
            float ry = (lane < HG_WARPS) ? s_y[lane] : -INFINITY;
            head_warp_combine<SAMPLE>(rm, rs, ri, rk, ry);
            if (np == 1) {
                const TileMeta mt{slot, 0, 0, st, lo, deg, 0};
                finalize_row(f, head_view(f), nullptr, mt, rm, rs, ri, lane, true, SAMPLE, ry);
            } else if (lane == 0) {
                a.gpartials[(long long)g * HG_MAX_PIECES + p] = HeadPartial{rm, rs, ri, rk, ry, {0, 0, 0}};
            }
        }
    }
}

// Gathered rows cut into several pieces: one warp per row merges the piece results in a fixed order (lane l takes
// the pieces l, l + 32, ascending, then the butterfly), then the CSR transition and the accept test.
template <bool SAMPLE>
__global__ void head_gather_finish_kernel(const HeadArgs a) {
    pdl_launch_dependents();  // launched with programmatic stream serialization: the next kernel may be scheduled,
    pdl_wait();               // and nothing of this one touches global memory before its predecessor has completed
    const StepArgs& f = a.fin;
    const int n_gather = __ldcg(a.hctr + 1);
    const int lane = threadIdx.x & 31;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int nwarps = (gridDim.x * blockDim.x) >> 5;
    for (int g = warp; g < n_gather; g += nwarps) {
        const int slot = __ldcg(a.gather_slot + g);
        const int st = __ldcg(a.gather_state + g);
        const long long lo = __ldg(f.dfa.row_ptr + st);
        const int deg = (int)(__ldg(f.dfa.row_ptr + st + 1) - lo);
        const int np = hg_pieces(deg);
        if (np == 1) continue;  // finished by its gather CTA
        float m = -INFINITY, s = 0.0f, kb = -INFINITY, yb = -INFINITY;
        int idx = 0x7FFFFFFF;
        for (int q = lane; q < np; q += 32) {
            const int4* pp = reinterpret_cast<const int4*>(a.gpartials + (long long)g * HG_MAX_PIECES + q);
            const int4 p = __ldcg(pp);
            if (SAMPLE) {
                const int4 p2 = __ldcg(pp + 1);
                int dummy = 0;
                online_combine(m, s, dummy, __int_as_float(p.x), __int_as_float(p.y), 0);
                head_sample_combine(kb, idx, yb, __int_as_float(p.w), p.z, __int_as_float(p2.x));
            } else {
                online_combine(m, s, idx, __int_as_float(p.x), __int_as_float(p.y), p.z);
            }
        }
        head_warp_combine<SAMPLE>(m, s, idx, kb, yb);
        const TileMeta mt{slot, 0, 0, st, lo, deg, 0};
        finalize_row(f, head_view(f), nullptr, mt, m, s, idx, lane, true, SAMPLE, yb);
    }
}

// ---------------------------------------------------------------- dense: tcgen05 contraction
// Persistent kernel, one CTA per SM.  Barriers:
//   full[s]  / empty[s]   shared-memory stage s: TMA -> MMA / MMA (tcgen05.commit) -> TMA
//   tfull[b] / tempty[b]  accumulator buffer b (256 TMEM columns): MMA -> epilogue / back
// Every role walks the same sequence (units of this CTA -> vocabulary tiles -> K blocks), so
// stage and phase counters stay in step without any other communication.
template <bool SAMPLE>
__global__ void __launch_bounds__(HD_THREADS, 1)
head_dense_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmW, const HeadArgs a) {
    pdl_launch_dependents();  // launched with programmatic stream serialization: the next kernel may be scheduled,
    pdl_wait();               // and nothing of this one touches global memory before its predecessor has completed
    extern __shared__ __align__(1024) unsigned char hd_smem[];
    __shared__ __align__(8) unsigned long long bar_full[HD_STAGES], bar_empty[HD_STAGES], bar_tfull[2], bar_tempty[2];
    __shared__ uint32_t s_tmem;

    const int n_dense = __ldcg(a.hctr + 0);
    if (a.pairs && n_dense >= HD2_MIN_ROWS) return;  // uniform: head_dense2_kernel (CTA pairs) runs this call
    const HeadSched hs = head_sched(n_dense, a.fin.dfa.V);
    if (hs.num_m == 0) return;  // uniform: nothing was allocated yet
    const int total_units = hs.num_m * hs.NU;
    const int num_k = (a.H + HD_BK - 1) / HD_BK;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t tiles = (smem_u32(hd_smem) + 1023u) & ~1023u;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmA);
        tma_prefetch_desc(&tmW);
#pragma unroll
        for (int s = 0; s < HD_STAGES; ++s) {
            mbar_init(smem_u32(&bar_full[s]), 1);
            mbar_init(smem_u32(&bar_empty[s]), 1);
        }
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            mbar_init(smem_u32(&bar_tfull[b]), 1);
            mbar_init(smem_u32(&bar_tempty[b]), 4);  // one arrival per epilogue warp
        }
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc(smem_u32(&s_tmem), HD_TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = s_tmem;

    if (warp == 0) {
        // ===== TMA producer (one lane)
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int u = blockIdx.x; u < total_units; u += gridDim.x) {
                const int m_tile = u % hs.num_m, n_unit = u / hs.num_m;
                const int nt0 = n_unit * hs.L, nt1 = min(nt0 + hs.L, hs.num_n);
                for (int nt = nt0; nt < nt1; ++nt) {
                    for (int kb = 0; kb < num_k; ++kb) {
                        mbar_wait(smem_u32(&bar_empty[stage]), phase ^ 1u);
                        const uint32_t bar = smem_u32(&bar_full[stage]);
                        const uint32_t sa = tiles + stage * HD_STAGE_BYTES;
                        mbar_arrive_expect_tx(bar, HD_STAGE_BYTES);
                        tma_load_2d(sa, &tmA, kb * HD_BK, m_tile * HD_BM, bar);
                        tma_load_2d(sa + HD_A_BYTES, &tmW, kb * HD_BK, nt * HD_BN, bar);
                        if (++stage == HD_STAGES) {
                            stage = 0;
                            phase ^= 1u;
                        }
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (one lane)
        if (lane == 0) {
            constexpr uint32_t idesc = umma_idesc_bf16(HD_BM, HD_BN);
            int stage = 0, ab = 0;
            uint32_t phase = 0, aphase = 0;
            for (int u = blockIdx.x; u < total_units; u += gridDim.x) {
                const int n_unit = u / hs.num_m;
                const int nt0 = n_unit * hs.L, nt1 = min(nt0 + hs.L, hs.num_n);
                for (int nt = nt0; nt < nt1; ++nt) {
                    mbar_wait(smem_u32(&bar_tempty[ab]), aphase ^ 1u);  // epilogue drained this buffer
                    tc_fence_after();
                    const uint32_t d_tmem = tmem + (uint32_t)ab * HD_BN;
                    for (int kb = 0; kb < num_k; ++kb) {
                        mbar_wait(smem_u32(&bar_full[stage]), phase);
                        tc_fence_after();
                        const uint32_t sa = tiles + stage * HD_STAGE_BYTES;
                        const uint64_t da = umma_desc_k_sw128(sa), db = umma_desc_k_sw128(sa + HD_A_BYTES);
#pragma unroll
                        for (int k = 0; k < HD_BK / HD_UK; ++k)
                            tc_mma_bf16(d_tmem, da + 2ull * k, db + 2ull * k, idesc, (kb | k) ? 1u : 0u);
                        tc_commit(smem_u32(&bar_empty[stage]));  // stage free once these MMAs have read it
                        if (++stage == HD_STAGES) {
                            stage = 0;
                            phase ^= 1u;
                        }
                    }
                    tc_commit(smem_u32(&bar_tfull[ab]));  // accumulator complete
                    ab ^= 1;
                    if (ab == 0) aphase ^= 1u;
                }
            }
        }
    } else {
        // ===== epilogue: thread <-> accumulator row (TMEM lane); a warp may only touch the lane
        // quadrant warp_id % 4
        const int quad = warp & 3;
        const int row_in_tile = quad * 32 + lane;
        const DfaDev& dfa = a.fin.dfa;
        int ab = 0;
        uint32_t aphase = 0;
        for (int u = blockIdx.x; u < total_units; u += gridDim.x) {
            const int m_tile = u % hs.num_m, n_unit = u / hs.num_m;
            const int nt0 = n_unit * hs.L, nt1 = min(nt0 + hs.L, hs.num_n);
            const int drow = m_tile * HD_BM + row_in_tile;
            const bool valid = drow < n_dense;
            const int st = valid ? __ldcg(a.dense_state + drow) : 0;
            const uint32_t* mrow = dfa.mask + (long long)st * dfa.Wpad;
            float m = -INFINITY, s = 0.0f, kb = -INFINITY, yb = -INFINITY;
            int idx = 0x7FFFFFFF;
            uint32_t row_key = 0u;
            if (SAMPLE && valid) {
                const int slot = __ldcg(a.dense_slot + drow);
                row_key = rng_row_key(a.fin.seed_lo, a.fin.seed_hi,
                                      (uint32_t)(a.fin.row_map ? __ldg(a.fin.row_map + slot) : slot),
                                      (uint32_t)(a.fin.rng_step_base + a.fin.step));
            }
            for (int nt = nt0; nt < nt1; ++nt) {
                const int n0 = nt * HD_BN;
                // the 8 mask words of this row for the tile's 256 tokens (two 16-byte loads)
                uint32_t mw[8];
                {
                    const int w0 = n0 >> 5;
                    uint4 lo4 = make_uint4(0, 0, 0, 0), hi4 = make_uint4(0, 0, 0, 0);
                    if (valid && w0 + 3 < dfa.Wpad) lo4 = __ldg(reinterpret_cast<const uint4*>(mrow + w0));
                    if (valid && w0 + 7 < dfa.Wpad) hi4 = __ldg(reinterpret_cast<const uint4*>(mrow + w0 + 4));
                    mw[0] = lo4.x; mw[1] = lo4.y; mw[2] = lo4.z; mw[3] = lo4.w;
                    mw[4] = hi4.x; mw[5] = hi4.y; mw[6] = hi4.z; mw[7] = hi4.w;
                }
                mbar_wait(smem_u32(&bar_tfull[ab]), aphase);
                tc_fence_after();
                const uint32_t tbase = tmem + ((uint32_t)(quad * 32) << 16) + (uint32_t)ab * HD_BN;
#pragma unroll
                for (int c = 0; c < HD_BN / 32; ++c) {
                    const uint32_t bits = mw[c];
                    if (__any_sync(FULL, bits != 0u)) {  // warp-uniform: skip columns nobody allows
                        uint32_t v[32];
                        tmem_ld32(tbase + c * 32, v);
                        tmem_ld_wait();
#pragma unroll
                        for (int j = 0; j < 32; ++j)
                            if ((bits >> j) & 1u) {
                                if (SAMPLE)
                                    head_update_sample(m, s, kb, idx, yb, fmaxf(__uint_as_float(v[j]), -INFINITY),
                                                       n0 + c * 32 + j, n0 + c * 32 + j, a.fin.inv_tau, row_key);
                                else
                                    online_update(m, s, idx, fmaxf(__uint_as_float(v[j]), -INFINITY), n0 + c * 32 + j);
                            }
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&bar_tempty[ab]));
                ab ^= 1;
                if (ab == 0) aphase ^= 1u;
            }
            if (valid) a.partials[(long long)drow * hs.NU + n_unit] = HeadPartial{m, s, idx, kb, yb, {0, 0, 0}};
        }
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    if (warp == 1) tmem_dealloc(tmem, HD_TMEM_COLS);
}

// ---------------------------------------------------------------- dense, CTA pairs (cta_group::2)
// The same contraction on pairs of SMs (thread-block cluster of 2, tcgen05.mma.cta_group::2, UMMA 256 x 256 x 16):
// a pair owns a tile of 256 rows x 256 tokens.  Per k-block each CTA loads ITS 128 rows of A and ITS 128 tokens of
// the W tile (32 KiB instead of 48 KiB: the tensor cores of both SMs read both halves of W), so the shared-memory
// ring holds 6 stages instead of 4 (2.3 us of look-ahead instead of 1.5) and the L2 -> SM operand traffic drops by a
// third.  Only the leader (cluster rank 0) issues MMAs; each CTA keeps the accumulator rows of its own 128 rows in
// its own TMEM and runs the same masked online-softmax epilogue as head_dense_kernel.
//   full[s]   (leader's): both producers' bytes (the TMA loads name the leader's barrier) + one arrival from each
//   empty[s]  (own): tcgen05.commit multicast to both CTAs
//   tfull[b]  (own): tcgen05.commit multicast;  tempty[b] (leader's): 4 epilogue warps of each CTA
// Used when more than 128 rows are dense (two row tiles or more); head_dense_kernel keeps the single-tile case.
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// one arrival on the mbarrier at the same shared-memory offset in CTA `cta` of the cluster
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t bar, uint32_t cta) {
    asm volatile(
        "{\n\t"
        ".reg .b32 r;\n\t"
        "mapa.shared::cluster.u32 r, %0, %1;\n\t"
        "mbarrier.arrive.shared::cluster.b64 _, [r];\n\t"
        "}" ::"r"(bar),
        "r"(cta)
        : "memory");
}
constexpr uint32_t PEER_BIT_MASK = 0xFEFFFFFFu;  // clears the bit that tells the two CTAs of a pair apart: the leader's copy
// 2-D tiled TMA load into THIS CTA's shared memory whose bytes complete on the LEADER's mbarrier
__device__ __forceinline__ void tma_load_2d_pair(uint32_t dst, const void* tmap, int c0, int c1, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
        "l"(reinterpret_cast<uint64_t>(tmap)), "r"(c0), "r"(c1), "r"(bar & PEER_BIT_MASK)
        : "memory");
}
__device__ __forceinline__ void tmem_alloc_pair(uint32_t smem_dst, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_pair(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
// one arrival on the mbarrier at this offset in BOTH CTAs once every MMA issued so far has completed
__device__ __forceinline__ void tc_commit_pair(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
                 "h"((uint16_t)3)
                 : "memory");
}
__device__ __forceinline__ void tc_mma_bf16_pair(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                                 uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}

template <bool SAMPLE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(HD_THREADS, 1)
head_dense2_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmWh, const HeadArgs a) {
    pdl_launch_dependents();  // launched with programmatic stream serialization: the next kernel may be scheduled,
    pdl_wait();               // and nothing of this one touches global memory before its predecessor has completed
    extern __shared__ __align__(1024) unsigned char hd_smem[];
    __shared__ __align__(8) unsigned long long bar_full[HD2_STAGES], bar_empty[HD2_STAGES], bar_tfull[2], bar_tempty[2];
    __shared__ uint32_t s_tmem;

    const int n_dense = __ldcg(a.hctr + 0);
    if (n_dense < HD2_MIN_ROWS) return;  // uniform over the grid: head_dense_kernel runs this call
    const HeadSched hs = head_sched2(n_dense, a.fin.dfa.V);
    const int total_units = hs.num_m * hs.NU;
    const int num_k = (a.H + HD_BK - 1) / HD_BK;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const int cluster_id = blockIdx.x >> 1, num_clusters = gridDim.x >> 1;
    const uint32_t tiles = (smem_u32(hd_smem) + 1023u) & ~1023u;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmA);
        tma_prefetch_desc(&tmWh);
#pragma unroll
        for (int s = 0; s < HD2_STAGES; ++s) {
            mbar_init(smem_u32(&bar_full[s]), 2);   // one arrival per producer (the peer's arrives remotely)
            mbar_init(smem_u32(&bar_empty[s]), 1);  // tcgen05.commit, multicast
        }
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            mbar_init(smem_u32(&bar_tfull[b]), 1);
            mbar_init(smem_u32(&bar_tempty[b]), 8);  // four epilogue warps of each CTA (leader's copy is the one waited on)
        }
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc_pair(smem_u32(&s_tmem), HD_TMEM_COLS);
    tc_fence_before();
    cluster_sync_all();  // barriers initialised and TMEM allocated in both CTAs before anyone signals the other
    tc_fence_after();
    const uint32_t tmem = s_tmem;

    if (warp == 0) {
        // ===== TMA producer (one lane, in both CTAs): its 128 rows of A, its 128 tokens of the W tile
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int u = cluster_id; u < total_units; u += num_clusters) {
                const int m_pair = u % hs.num_m, n_unit = u / hs.num_m;
                const int nt0 = n_unit * hs.L, nt1 = min(nt0 + hs.L, hs.num_n);
                for (int nt = nt0; nt < nt1; ++nt) {
                    for (int kb = 0; kb < num_k; ++kb) {
                        mbar_wait(smem_u32(&bar_empty[stage]), phase ^ 1u);
                        const uint32_t bar = smem_u32(&bar_full[stage]);
                        const uint32_t sa = tiles + stage * HD2_STAGE_BYTES;
                        if (rank == 0) mbar_arrive_expect_tx(bar, 2 * HD2_STAGE_BYTES);
                        else mbar_arrive_cluster(bar, 0);
                        tma_load_2d_pair(sa, &tmA, kb * HD_BK, m_pair * 2 * HD_BM + (int)rank * HD_BM, bar);
                        tma_load_2d_pair(sa + HD_A_BYTES, &tmWh, kb * HD_BK, nt * HD_BN + (int)rank * HD2_HALF_N, bar);
                        if (++stage == HD2_STAGES) {
                            stage = 0;
                            phase ^= 1u;
                        }
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (one lane of the leader)
        if (lane == 0 && rank == 0) {
            constexpr uint32_t idesc = umma_idesc_bf16(2 * HD_BM, HD_BN);
            int stage = 0, ab = 0;
            uint32_t phase = 0, aphase = 0;
            for (int u = cluster_id; u < total_units; u += num_clusters) {
                const int n_unit = u / hs.num_m;
                const int nt0 = n_unit * hs.L, nt1 = min(nt0 + hs.L, hs.num_n);
                for (int nt = nt0; nt < nt1; ++nt) {
                    mbar_wait(smem_u32(&bar_tempty[ab]), aphase ^ 1u);  // both epilogues drained this buffer
                    tc_fence_after();
                    const uint32_t d_tmem = tmem + (uint32_t)ab * HD_BN;
                    for (int kb = 0; kb < num_k; ++kb) {
                        mbar_wait(smem_u32(&bar_full[stage]), phase);
                        tc_fence_after();
                        const uint32_t sa = tiles + stage * HD2_STAGE_BYTES;
                        const uint64_t da = umma_desc_k_sw128(sa), db = umma_desc_k_sw128(sa + HD_A_BYTES);
#pragma unroll
                        for (int k = 0; k < HD_BK / HD_UK; ++k)
                            tc_mma_bf16_pair(d_tmem, da + 2ull * k, db + 2ull * k, idesc, (kb | k) ? 1u : 0u);
                        tc_commit_pair(smem_u32(&bar_empty[stage]));  // stage free in both CTAs once these MMAs have read it
                        if (++stage == HD2_STAGES) {
                            stage = 0;
                            phase ^= 1u;
                        }
                    }
                    tc_commit_pair(smem_u32(&bar_tfull[ab]));  // accumulator complete, both halves
                    ab ^= 1;
                    if (ab == 0) aphase ^= 1u;
                }
            }
        }
    } else {
        // ===== epilogue (both CTAs): thread <-> accumulator row of this CTA's 128 rows
        const int quad = warp & 3;
        const int row_in_tile = quad * 32 + lane;
        const DfaDev& dfa = a.fin.dfa;
        int ab = 0;
        uint32_t aphase = 0;
        for (int u = cluster_id; u < total_units; u += num_clusters) {
            const int m_pair = u % hs.num_m, n_unit = u / hs.num_m;
            const int nt0 = n_unit * hs.L, nt1 = min(nt0 + hs.L, hs.num_n);
            const int drow = m_pair * 2 * HD_BM + (int)rank * HD_BM + row_in_tile;
            const bool valid = drow < n_dense;
            const int st = valid ? __ldcg(a.dense_state + drow) : 0;
            const uint32_t* mrow = dfa.mask + (long long)st * dfa.Wpad;
            float m = -INFINITY, s = 0.0f, kb = -INFINITY, yb = -INFINITY;
            int idx = 0x7FFFFFFF;
            uint32_t row_key = 0u;
            if (SAMPLE && valid) {
                const int slot = __ldcg(a.dense_slot + drow);
                row_key = rng_row_key(a.fin.seed_lo, a.fin.seed_hi,
                                      (uint32_t)(a.fin.row_map ? __ldg(a.fin.row_map + slot) : slot),
                                      (uint32_t)(a.fin.rng_step_base + a.fin.step));
            }
            for (int nt = nt0; nt < nt1; ++nt) {
                const int n0 = nt * HD_BN;
                uint32_t mw[8];
                {
                    const int w0 = n0 >> 5;
                    uint4 lo4 = make_uint4(0, 0, 0, 0), hi4 = make_uint4(0, 0, 0, 0);
                    if (valid && w0 + 3 < dfa.Wpad) lo4 = __ldg(reinterpret_cast<const uint4*>(mrow + w0));
                    if (valid && w0 + 7 < dfa.Wpad) hi4 = __ldg(reinterpret_cast<const uint4*>(mrow + w0 + 4));
                    mw[0] = lo4.x; mw[1] = lo4.y; mw[2] = lo4.z; mw[3] = lo4.w;
                    mw[4] = hi4.x; mw[5] = hi4.y; mw[6] = hi4.z; mw[7] = hi4.w;
                }
                mbar_wait(smem_u32(&bar_tfull[ab]), aphase);
                tc_fence_after();
                const uint32_t tbase = tmem + ((uint32_t)(quad * 32) << 16) + (uint32_t)ab * HD_BN;
#pragma unroll
                for (int c = 0; c < HD_BN / 32; ++c) {
                    const uint32_t bits = mw[c];
                    if (__any_sync(FULL, bits != 0u)) {  // warp-uniform: skip columns nobody allows
                        uint32_t v[32];
                        tmem_ld32(tbase + c * 32, v);
                        tmem_ld_wait();
#pragma unroll
                        for (int j = 0; j < 32; ++j)
                            if ((bits >> j) & 1u) {
                                if (SAMPLE)
                                    head_update_sample(m, s, kb, idx, yb, fmaxf(__uint_as_float(v[j]), -INFINITY),
                                                       n0 + c * 32 + j, n0 + c * 32 + j, a.fin.inv_tau, row_key);
                                else
                                    online_update(m, s, idx, fmaxf(__uint_as_float(v[j]), -INFINITY), n0 + c * 32 + j);
                            }
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(smem_u32(&bar_tempty[ab]), 0);  // the leader's barrier
                ab ^= 1;
                if (ab == 0) aphase ^= 1u;
            }
            if (valid) a.partials[(long long)drow * hs.NU + n_unit] = HeadPartial{m, s, idx, kb, yb, {0, 0, 0}};
        }
    }
    tc_fence_before();
    cluster_sync_all();  // nobody leaves (or frees TMEM) while the other CTA may still read its shared memory / signal it
    tc_fence_after();
    if (warp == 1) tmem_dealloc_pair(tmem, HD_TMEM_COLS);
}

// ---------------------------------------------------------------- finish dense rows
// One warp per dense row: partials merged in a fixed order (lane q % 32 takes ranges q, q + 32,
// ... ascending, then the butterfly), then the CSR transition and the accept test.
template <bool SAMPLE>
__global__ void head_finish_kernel(const HeadArgs a) {
    pdl_launch_dependents();  // launched with programmatic stream serialization: the next kernel may be scheduled,
    pdl_wait();               // and nothing of this one touches global memory before its predecessor has completed
    const StepArgs& f = a.fin;
    const int n_dense = __ldcg(a.hctr + 0);
    const int NU = head_row_partials(n_dense, f.dfa.V, a.pairs);
    const int lane = threadIdx.x & 31;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int nwarps = (gridDim.x * blockDim.x) >> 5;
    for (int d = warp; d < n_dense; d += nwarps) {
        const int slot = __ldcg(a.dense_slot + d);
        const int st = __ldcg(a.dense_state + d);
        float m = -INFINITY, s = 0.0f, kb = -INFINITY, yb = -INFINITY;
        int idx = 0x7FFFFFFF;
        for (int q = lane; q < NU; q += 32) {
            const int4* pp = reinterpret_cast<const int4*>(a.partials + (long long)d * NU + q);
            const int4 p = __ldcg(pp);
            if (SAMPLE) {
                const int4 p2 = __ldcg(pp + 1);
                int dummy = 0;
                online_combine(m, s, dummy, __int_as_float(p.x), __int_as_float(p.y), 0);
                head_sample_combine(kb, idx, yb, __int_as_float(p.w), p.z, __int_as_float(p2.x));
            } else {
                online_combine(m, s, idx, __int_as_float(p.x), __int_as_float(p.y), p.z);
            }
        }
        head_warp_combine<SAMPLE>(m, s, idx, kb, yb);
        const long long lo = __ldg(f.dfa.row_ptr + st);
        const int deg = (int)(__ldg(f.dfa.row_ptr + st + 1) - lo);
        const TileMeta mt{slot, 0, 0, st, lo, deg, 0};
        finalize_row(f, head_view(f), nullptr, mt, m, s, idx, lane, false, SAMPLE, yb);
    }
}

// ---------------------------------------------------------------- decode loop: compaction
// Last kernel of a loop step: stable early-exit compaction of the active list.
__global__ void __launch_bounds__(1024, 1) head_loop_tail_kernel(const HeadArgs a) {
    pdl_launch_dependents();  // launched with programmatic stream serialization: the next kernel may be scheduled,
    pdl_wait();               // and nothing of this one touches global memory before its predecessor has completed
    const StepArgs& f = a.fin;
    const int n = f.n_dev ? __ldcg(f.n_dev) : f.n;
    block_compact(f.done_out, f.row_map, f.state, n, f.cmp_row_ids_out, f.cmp_state_out, f.cmp_n_out);
    // LIMIT early exit: enough rows satisfied -> every row still active is cancelled
    if (f.sat_ctr && threadIdx.x == 0 && __ldcg(f.sat_ctr) >= f.limit) *f.cmp_n_out = 0;
}

}  // namespace cd
