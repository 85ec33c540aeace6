// cd_step.cuh -- the fused constrained step (include/cd.h cd_step).
//
// Design (B200-first; the paper gives no kernel):
//   * The step is one streaming pass over the logits, so it is HBM-bound: the job is to keep
//     enough bytes in flight and to waste no issue slots.  Every WARP owns a private ring of
//     STAGES shared-memory slots that it fills itself with 1-D bulk async copies (TMA engine,
//     cp.async.bulk -> SASS UBLKCP) completing on per-slot mbarriers: a logits tile and the
//     matching piece of the state's allowed-token bitmask land together.  No register staging,
//     no block-wide barriers in the streaming phase, WARPS*STAGES*TILE_BYTES in flight per SM.
//   * Work unit = (active slot, part of the row).  Units are handed out by one global atomic
//     counter (dynamic balance across the 148 SMs; the two dies do not run at the same speed);
//     the number of tiles per unit is derived on the device from the number of active rows, so
//     the same launch shape serves a full batch and the few-rows tail of an early-exit loop
//     without any host read of the active count.
//   * Per tile a lane walks the set bits of its mask words (warp-uniform trip count, branch
//     free body) and updates an online (max, sum-exp, argmax) triple; only allowed elements
//     cost arithmetic.
//   * Unit results of a row are merged without any fence: a unit stores its result into a slot
//     of three 64-bit words, each carrying the launch generation in its upper half (8-byte
//     stores are single-copy atomic, so a word is either stale or complete), then takes a
//     RELAXED ticket.  The warp that draws the last ticket merges: it reads the other slots and
//     re-reads any word whose tag is not current yet (the writers issued those stores before
//     their tickets, so they are on their way; normally the first read succeeds).  A
//     __threadfence here cost 3.8 us per unit (profiles/r1b): it waits for the bulk copies the
//     same warp still has in flight.
//   * That warp also does the CSR transition (128-ary warp search; row bounds were prefetched
//     into the tile meta, accepting[next] rides in bit 31 of next[]), the output writes and, in
//     the decode loop, the per-row history, while the other warps keep streaming.
//   * The last CTA to finish resets the work counter, bumps the generation and, in the decode
//     loop, performs the stable early-exit compaction: one launch per decoding step.
//   * Density-adaptive rows (GATHER instantiation): a row whose state has at most
//     `gather_max` transitions is not scanned at all -- its units walk pieces of the state's CSR
//     token list (coalesced) and gather exactly the allowed logits (one 32-byte sector each, 8
//     independent loads per lane in flight).  The running argmax is the CSR position, so the
//     transition needs no search.  Same outputs as the dense scan; dense and gathered rows mix
//     freely in one launch and share the merge / compaction machinery.
#pragma once
#include "cd_common.cuh"

namespace cd {

constexpr int TPU_MAX_BYTES = 65536;  // at most 64 KiB of logits per unit
constexpr int UNITS_PER_WARP = 4;     // aim for >= 4 units per warp when rows are few

constexpr int FLAG_FIRST = 1;   // first tile of its unit: reset the lane accumulators
constexpr int FLAG_LAST = 2;    // last tile of its unit: reduce and publish
constexpr int FLAG_ACCEPT = 4;  // pseudo tile of a slot whose state already accepts (no copy)
constexpr int FLAG_BADSTATE = 8;
constexpr int FLAG_GATHER = 16;  // pseudo tile of a gathered row piece (no copy); meta.tile = logits row

constexpr int SAMPLE_LIST_CAP = 128;  // tiles with at most this many allowed elements are compacted (SAMPLE)

constexpr int GATHER_CHUNK = 256;  // a gathered row is split into pieces of >= this many transitions
constexpr int GATHER_UNROLL = 8;   // independent gathers per lane in flight

// number of units a gathered row of `len` transitions is split into (P = units per row of the launch)
__host__ __device__ inline int gather_parts(int len, int P) {
    int np = (len + GATHER_CHUNK - 1) / GATHER_CHUNK;
    if (np < 1) np = 1;
    return np < P ? np : P;
}

// Result of one unit, readable without a fence: {gen:32 | payload:32} x 3 (+ pad to 32 B).
struct __align__(32) PartialSlot {
    unsigned long long m, s, idx, pad;
};

struct StepArgs {
    DfaDev dfa;
    const unsigned char* logits;
    long long ld_bytes;
    const int* row_map;
    int* state;      // [n] in: state of every slot (read-only while units are in flight); out: next state
    int* state_new;  // [n] scratch: next states, moved to `state` (or compacted) by the last CTA
    int n;
    const int* n_dev;  // if non-null the active count is read from the device
    int* token_out;
    float* logprob_out;
    float* lse_out;
    uint8_t* done_out;
    // scratch (per handle+stream)
    PartialSlot* partials;  // [units]
    int* tickets;           // [rows] arrivals per slot, zero between launches
    int* ctrs;              // [0] work counter, [1] finished CTAs, [2] sticky error count, [3] generation
    int gather_max;         // states with <= gather_max transitions are gathered (GATHER kernels; 0 = never)
    int all_gather;         // no state has more than gather_max transitions
    // decode loop only, all optional:
    // per-row history, indexed by ORIGINAL row id (= row_map[slot]), written when the row's step is final
    int* hist_tokens;  // [B, max_steps]
    int* hist_len;
    int* hist_final_state;
    float* hist_sum_logprob;
    uint8_t* hist_done;
    int step, max_steps;
    // fused early-exit compaction by the last CTA: (row_map, state) of not-done slots -> out lists
    int* cmp_row_ids_out;
    int* cmp_state_out;
    int* cmp_n_out;
    // LIMIT early exit (PAPER.md 2.4 "Early Exiting"), optional: rows that finish in a
    // state with satisfying[s] != 0 are counted in *sat_ctr; once it reaches `limit` the last CTA
    // empties the active list (every row still active is cancelled)
    const uint8_t* satisfying;  // [S]
    int* sat_ctr;
    int limit;
    // sampling (SAMPLE instantiation): Gumbel-max at temperature 1 / inv_tau with the
    // counter-based noise of (seed, original row id, rng_step_base + step, token)
    float inv_tau;
    uint32_t seed_lo, seed_hi;
    int rng_step_base;
    // host-buffer loop: the logits buffer holds the ACTIVE rows only, row = slot (row_map still names
    // the original row for the history and the sampling noise)
    int logits_by_slot;
    int upw, tpu_max;  // unit sizing (tuning knobs CD_UPW / CD_TPU_MAX): target units per warp, most tiles per unit
};

struct __align__(16) TileMeta {
    int slot;
    int tile;   // tile index inside the row
    int flags;  // FLAG_* | part << 8
    int st;     // automaton state of the slot
    long long csr_lo;  // row_ptr[st]
    int csr_len;       // row_ptr[st + 1] - row_ptr[st]
    int pad;
};

template <int STAGES, int TILE_BYTES>
struct __align__(128) WarpRing {
    unsigned char logits[STAGES][TILE_BYTES];
    unsigned char mask[STAGES][TILE_BYTES / 16];  // bf16: TILE_BYTES/2 tokens / 8; fp32 uses half
    TileMeta meta[STAGES];
    unsigned long long bar[STAGES];
    unsigned short list[SAMPLE_LIST_CAP];  // SAMPLE: positions of a tile's allowed elements, compacted
};

// tiles per unit for n active rows (host mirrors this in cd_api.cu: step_units_cap)
__host__ __device__ inline int tiles_per_unit(long long n, int tiles_per_row, long long total_warps, int tpu_max,
                                              int upw = UNITS_PER_WARP) {
    long long t = (n * tiles_per_row + total_warps * upw - 1) / (total_warps * upw);
    if (t < 1) t = 1;
    if (t > tpu_max) t = tpu_max;
    return (int)t;
}

template <int DT>
__device__ __forceinline__ float tile_elem(const unsigned char* tile, int e) {
    float x;
    if (DT == DT_BF16) {
        x = __uint_as_float(((uint32_t) reinterpret_cast<const uint16_t*>(tile)[e]) << 16);
    } else {
        x = reinterpret_cast<const float*>(tile)[e];
    }
    return fmaxf(x, -INFINITY);  // NaN -> -inf
}

// Row finished: (m, s, idx) is the merged result of all its units.  Warp-uniform.
// `gathered`: idx is the position inside the state's CSR row instead of the token id.
// `sampled`: idx is the sampled token (position), ytok its tempered logit: logprob = (ytok - m) - log(sum).
__device__ __forceinline__ void finalize_row(const StepArgs& a, const TileMeta& mt, float m, float s, int idx,
                                             int lane, bool gathered, bool sampled = false, float ytok = 0.0f) {
    const long long lo = mt.csr_lo, hi = mt.csr_lo + mt.csr_len;
    int token;
    float lp, lse;
    long long j;
    if (m == -INFINITY) {  // every allowed logit is -inf: lowest allowed id (G6)
        token = __ldg(a.dfa.tok + lo);
        lp = -INFINITY;
        lse = -INFINITY;
        idx = 0;
    } else {
        token = idx;
        const float L = logf(s);
        lp = sampled ? (ytok - m) - L : -L;  // greedy: log p(t*) = -log(sum); never m - lse (cancellation)
        lse = m + L;
    }
    if (gathered) {
        j = lo + idx;
        token = __ldg(a.dfa.tok + j);
    } else {
        j = warp_csr_find(a.dfa.tok, lo, hi, token, lane);
    }
    if (lane == 0) {
        const int slot = mt.slot;
        int ns = mt.st;
        uint8_t dn;
        if (j >= 0) {
            const int packed = __ldg(a.dfa.next + j);  // next state | accepting << 31
            ns = packed & 0x7FFFFFFF;
            dn = (packed < 0) ? 1 : 0;
        } else {
            atomicAdd(a.ctrs + 2, 1);
            dn = 1;
        }
        a.state_new[slot] = ns;
        a.token_out[slot] = token;
        a.logprob_out[slot] = lp;
        if (a.lse_out) a.lse_out[slot] = lse;
        a.done_out[slot] = dn;
        if (a.hist_tokens) {  // decode loop: this slot's row, original id
            const long long rid = a.row_map ? __ldg(a.row_map + slot) : slot;
            a.hist_tokens[rid * a.max_steps + a.step] = token;
            a.hist_len[rid] = a.step + 1;
            a.hist_final_state[rid] = ns;
            a.hist_sum_logprob[rid] += lp;
            a.hist_done[rid] = dn;
            if (a.sat_ctr && dn && __ldg(a.satisfying + ns)) atomicAdd(a.sat_ctr, 1);
        }
    }
}

template <bool SAMPLE>
__device__ __forceinline__ void warp_combine_s(float& m, float& s, int& idx, float& kb) {
    if constexpr (!SAMPLE) {
        warp_combine(m, s, idx);
    } else {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float m2 = __shfl_xor_sync(FULL, m, o);
            const float s2 = __shfl_xor_sync(FULL, s, o);
            const int i2 = __shfl_xor_sync(FULL, idx, o);
            const float k2 = __shfl_xor_sync(FULL, kb, o);
            int dummy = 0;
            online_combine(m, s, dummy, m2, s2, 0);
            sample_combine(kb, idx, k2, i2);
        }
    }
}

template <int DT, int WARPS, int STAGES, int TILE_BYTES, bool GATHER, bool SAMPLE = false>
__global__ void __launch_bounds__(WARPS * 32, 1) step_kernel(const StepArgs a) {
    constexpr int SZ = (DT == DT_BF16) ? 2 : 4;
    constexpr int TILE_TOK = TILE_BYTES / SZ;
    constexpr int MASK_BYTES = TILE_TOK / 8;
    constexpr int WPL = TILE_TOK / 1024;  // mask words per lane and tile
    constexpr int TPU_MAX = TPU_MAX_BYTES / TILE_BYTES;
    static_assert(WPL >= 1 && TILE_TOK % 1024 == 0, "tile must hold a multiple of 32 mask words");
    using Ring = WarpRing<STAGES, TILE_BYTES>;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    Ring& ring = reinterpret_cast<Ring*>(smem_raw)[warp];

    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) mbar_init(smem_u32(&ring.bar[s]), 1);
        fence_mbar_init();
    }
    __syncwarp();

    // Programmatic dependent launch: the next step's grid may be scheduled as soon as every CTA
    // of this one got here (its CTAs land on SMs as ours exit and set up their barriers), but
    // nothing of this kernel reads or writes global memory before the previous grid has
    // completed and flushed (griddepcontrol.wait).
    pdl_launch_dependents();
    pdl_wait();

    // ---------------- issue side (warp-uniform state)
    // The first unit of a warp is its global warp id (no atomic on the start-up chain); later
    // units come from the work counter, which therefore starts at 0 = unit `total_warps`.
    const int total_warps = gridDim.x * WARPS;
    int next_u_l0 = blockIdx.x * WARPS + warp;  // prefetched unit id, valid in lane 0
    const unsigned gen = (unsigned)__ldcg(a.ctrs + 3);  // launch generation (tag of the partial slots)
    const int n = a.n_dev ? __ldcg(a.n_dev) : a.n;
    const int V = a.dfa.V;
    const int tiles_per_row = (V + TILE_TOK - 1) / TILE_TOK;
    const int tpu = tiles_per_unit(n, tiles_per_row, total_warps, min(TPU_MAX, a.tpu_max), a.upw);
    const int Pd = (tiles_per_row + tpu - 1) / tpu;  // units per row of a dense scan
    // a gathered row is split only as far as needed to give every warp a few units
    const int PG = GATHER ? max(1, min(Pd, (total_warps * UNITS_PER_WARP) / max(n, 1))) : Pd;
    // units per row of this launch; if every state is gathered no unit is drawn in vain
    const int P = (GATHER && a.all_gather) ? PG : Pd;
    const int total_units = n * P;
    const bool ragged_row = (V % TILE_TOK) != 0;
    const uint64_t pol_stream = l2_policy_evict_first();

    bool exhausted = false;
    int iss_tile = 0, iss_end = 0;
    int iss_slot = 0, iss_st = 0, iss_flags = 0, iss_len = 0, iss_row = 0;
    long long iss_lo = 0;
    const unsigned char* iss_src = nullptr;  // next logits tile of the current unit
    const unsigned char* iss_msk = nullptr;  // next mask piece
    int iss_stage = 0, in_flight = 0;

    auto issue_one = [&]() {
        while (iss_tile >= iss_end) {  // next unit (units of a gathered row beyond its pieces are skipped)
            if (exhausted) return;
            const int u = __shfl_sync(FULL, next_u_l0, 0);
            if (u >= total_units) {
                exhausted = true;
                return;
            }
            if (lane == 0) next_u_l0 = total_warps + atomicAdd(a.ctrs + 0, 1);
            iss_slot = u / P;
            const int part = u - iss_slot * P;
            // state[] is not written while units are in flight (next states go to state_new[]): a
            // unit drawn after its row was finalised still sees the state the row was processed in
            iss_st = a.state[iss_slot];
            const long long r = a.row_map ? (long long)__ldg(a.row_map + iss_slot) : (long long)iss_slot;
            const long long rl = a.logits_by_slot ? (long long)iss_slot : r;  // row of the logits buffer
            iss_row = (int)rl;
            const bool bad = (iss_st < 0) || (iss_st >= a.dfa.S);
            const int sts = bad ? 0 : iss_st;
            const bool acc = !bad && (__ldg(a.dfa.accepting + sts) != 0);
            iss_lo = __ldg(a.dfa.row_ptr + sts);
            iss_len = (int)(__ldg(a.dfa.row_ptr + sts + 1) - iss_lo);
            if (bad || acc) {
                if (lane == 0) {
                    ring.meta[iss_stage] =
                        TileMeta{iss_slot, 0, (bad ? FLAG_BADSTATE : FLAG_ACCEPT) | (part << 8), iss_st, 0, 0, 0};
                    mbar_arrive(smem_u32(&ring.bar[iss_stage]));
                }
                iss_stage = (iss_stage + 1 == STAGES) ? 0 : iss_stage + 1;
                ++in_flight;
                iss_tile = iss_end = 0;
                return;
            }
            if (GATHER && iss_len <= a.gather_max) {
                if (part >= gather_parts(iss_len, PG)) continue;
                if (lane == 0) {
                    ring.meta[iss_stage] = TileMeta{iss_slot, (int)rl, FLAG_GATHER | FLAG_LAST | (part << 8), iss_st,
                                                    iss_lo, iss_len, 0};
                    mbar_arrive(smem_u32(&ring.bar[iss_stage]));
                }
                iss_stage = (iss_stage + 1 == STAGES) ? 0 : iss_stage + 1;
                ++in_flight;
                iss_tile = iss_end = 0;
                return;
            }
            iss_tile = part * tpu;
            iss_end = min(iss_tile + tpu, tiles_per_row);
            iss_src = a.logits + rl * a.ld_bytes + (long long)iss_tile * TILE_BYTES;
            iss_msk = reinterpret_cast<const unsigned char*>(a.dfa.mask + (long long)iss_st * a.dfa.Wpad) +
                      (long long)iss_tile * MASK_BYTES;
            iss_flags = (part << 8) | FLAG_FIRST;
        }
        const uint32_t bar = smem_u32(&ring.bar[iss_stage]);
        const uint32_t dst = smem_u32(ring.logits[iss_stage]);
        const uint32_t mdst = smem_u32(ring.mask[iss_stage]);
        const int fl = iss_flags | ((iss_tile + 1 == iss_end) ? FLAG_LAST : 0);
        if (ragged_row && iss_tile + 1 == tiles_per_row) {
            // last tile of a row whose length is not a multiple of the tile: partial copies; the
            // < 16 trailing logits bytes go through plain loads, unused mask words are zeroed.
            const int ntok = V - iss_tile * TILE_TOK;
            const uint32_t bytes = (uint32_t)ntok * SZ;
            const uint32_t bulk = bytes & ~15u;
            const uint32_t mbytes = (uint32_t)(((ntok + 31) >> 5) * 4 + 15) & ~15u;
            const int e = (int)(bulk / SZ) + lane;
            if (e < ntok) {
                if (DT == DT_BF16)
                    reinterpret_cast<uint16_t*>(ring.logits[iss_stage])[e] =
                        reinterpret_cast<const uint16_t*>(iss_src)[e];
                else
                    reinterpret_cast<float*>(ring.logits[iss_stage])[e] = reinterpret_cast<const float*>(iss_src)[e];
            }
            for (int w = (int)(mbytes / 4) + lane; w < MASK_BYTES / 4; w += 32)
                reinterpret_cast<uint32_t*>(ring.mask[iss_stage])[w] = 0u;
            __syncwarp();
            if (lane == 0) {
                ring.meta[iss_stage] = TileMeta{iss_slot, iss_tile, fl, iss_st, iss_lo, iss_len, iss_row};
                mbar_arrive_expect_tx(bar, bulk + mbytes);
                if (bulk) bulk_g2s_hint(dst, iss_src, bulk, bar, pol_stream);
                bulk_g2s(mdst, iss_msk, mbytes, bar);
            }
        } else if (lane == 0) {
            ring.meta[iss_stage] = TileMeta{iss_slot, iss_tile, fl, iss_st, iss_lo, iss_len, iss_row};
            mbar_arrive_expect_tx(bar, TILE_BYTES + MASK_BYTES);
            bulk_g2s_hint(dst, iss_src, TILE_BYTES, bar, pol_stream);
            bulk_g2s(mdst, iss_msk, MASK_BYTES, bar);
        }
        iss_flags &= ~FLAG_FIRST;
        iss_src += TILE_BYTES;
        iss_msk += MASK_BYTES;
        ++iss_tile;
        ++in_flight;
        iss_stage = (iss_stage + 1 == STAGES) ? 0 : iss_stage + 1;
    };

#pragma unroll 1
    for (int k = 0; k < STAGES; ++k) issue_one();

    // ---------------- consume side
    float m = -INFINITY, s = 0.0f, kb = -INFINITY;  // kb: best perturbed key (SAMPLE); idx then is its token
    int idx = 0x7FFFFFFF;
    const int rng_step = a.rng_step_base + a.step;
    int cons_stage = 0;
    uint32_t cons_phase = 0;
    const unsigned long long tag = (unsigned long long)gen << 32;

#pragma unroll 1
    while (in_flight > 0) {
        mbar_wait(smem_u32(&ring.bar[cons_stage]), cons_phase);
        __syncwarp();
        const TileMeta mt = ring.meta[cons_stage];
        const int part = mt.flags >> 8;

        if (mt.flags & (FLAG_ACCEPT | FLAG_BADSTATE)) {
            // accepted rows never advance
            if (part == 0 && lane == 0) {
                a.state_new[mt.slot] = mt.st;
                a.token_out[mt.slot] = -1;
                a.logprob_out[mt.slot] = 0.0f;
                if (a.lse_out) a.lse_out[mt.slot] = 0.0f;
                a.done_out[mt.slot] = 1;
                if (mt.flags & FLAG_BADSTATE) atomicAdd(a.ctrs + 2, 1);
            }
        } else {
            const bool gathered = GATHER && (mt.flags & FLAG_GATHER);
            const int np = gathered ? gather_parts(mt.csr_len, PG) : P;  // units this row was split into
            if (gathered) {
                // piece [j0, j1) of the state's CSR row: tokens read coalesced, their logits gathered
                // with GATHER_UNROLL independent loads per lane; idx = position in the CSR row, which
                // ascends with the token id, so "replace on strictly greater" keeps the lowest id
                m = -INFINITY;
                s = 0.0f;
                kb = -INFINITY;
                idx = 0x7FFFFFFF;
                const uint32_t row_key = SAMPLE ? rng_row_key(a.seed_lo, a.seed_hi, (uint32_t)(a.row_map ? __ldg(a.row_map + mt.slot) : mt.slot), (uint32_t)rng_step) : 0u;
                const int j0 = (int)(((long long)mt.csr_len * part) / np);
                const int j1 = (int)(((long long)mt.csr_len * (part + 1)) / np);
                const int* tk = a.dfa.tok + mt.csr_lo;
                const unsigned char* rowp = a.logits + (long long)mt.tile * a.ld_bytes;
                // software pipeline: the token ids of the next round are loaded while this round's
                // logits are in flight
                int t[GATHER_UNROLL];
#pragma unroll
                for (int u = 0; u < GATHER_UNROLL; ++u)
                    t[u] = (j0 + lane + 32 * u < j1) ? __ldg(tk + j0 + lane + 32 * u) : -1;
#pragma unroll 1
                for (int j = j0 + lane; j < j1; j += 32 * GATHER_UNROLL) {
                    float x[GATHER_UNROLL];
#pragma unroll
                    for (int u = 0; u < GATHER_UNROLL; ++u) {
                        float v = -INFINITY;
                        if (t[u] >= 0) {
                            if (DT == DT_BF16)
                                v = __uint_as_float(
                                    ((uint32_t)__ldg(reinterpret_cast<const uint16_t*>(rowp) + t[u])) << 16);
                            else
                                v = __ldg(reinterpret_cast<const float*>(rowp) + t[u]);
                        }
                        x[u] = v;
                    }
                    const int jn = j + 32 * GATHER_UNROLL;
                    int tc[GATHER_UNROLL];
#pragma unroll
                    for (int u = 0; u < GATHER_UNROLL; ++u) tc[u] = t[u];
#pragma unroll
                    for (int u = 0; u < GATHER_UNROLL; ++u) t[u] = (jn + 32 * u < j1) ? __ldg(tk + jn + 32 * u) : -1;
#pragma unroll
                    for (int u = 0; u < GATHER_UNROLL; ++u) {
                        if (SAMPLE)
                            online_update_sample(m, s, kb, idx, fmaxf(x[u], -INFINITY), tc[u], j + 32 * u, a.inv_tau, row_key);
                        else
                            online_update(m, s, idx, fmaxf(x[u], -INFINITY), j + 32 * u);  // NaN -> -inf
                    }
                }
                __syncwarp();
            } else {
            if (mt.flags & FLAG_FIRST) {
                m = -INFINITY;
                s = 0.0f;
                kb = -INFINITY;
                idx = 0x7FFFFFFF;
            }
            const uint32_t row_key = SAMPLE ? rng_row_key(a.seed_lo, a.seed_hi, (uint32_t)(a.row_map ? __ldg(a.row_map + mt.slot) : mt.slot), (uint32_t)rng_step) : 0u;
            const int t0 = mt.tile * TILE_TOK;
            const uint32_t* mw = reinterpret_cast<const uint32_t*>(ring.mask[cons_stage]);
            const unsigned char* tile = ring.logits[cons_stage];
            uint32_t bits[WPL];
#pragma unroll
            for (int j = 0; j < WPL; ++j) bits[j] = mw[j * 32 + lane];
            // SAMPLE, sparse tile: the noise costs ~60 instructions per evaluation, so the allowed
            // positions are first compacted across the warp (exclusive scan of the per-lane popcounts
            // in (word, lane) = ascending token order, positions written to a small shared list) and
            // each lane then evaluates exactly the elements of rank lane, lane + 32, ... (ascending per
            // lane, so "replace on strictly greater" still keeps the lowest id).
            bool compacted = false;
            if constexpr (SAMPLE) {
                int cnt[WPL], offs[WPL], total = 0;
#pragma unroll
                for (int j = 0; j < WPL; ++j) {
                    cnt[j] = __popc(bits[j]);
                    int inc = cnt[j];
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int up = __shfl_up_sync(FULL, inc, o);
                        if (lane >= o) inc += up;
                    }
                    offs[j] = total + inc - cnt[j];
                    total += __shfl_sync(FULL, inc, 31);
                }
                if (total <= SAMPLE_LIST_CAP) {
                    compacted = true;
#pragma unroll
                    for (int j = 0; j < WPL; ++j) {
                        uint32_t b = bits[j];
                        int o = offs[j];
                        const int e0 = (j * 32 + lane) * 32;
                        while (b != 0u) {
                            ring.list[o++] = (unsigned short)(e0 + __ffs(b) - 1);
                            b &= b - 1u;
                        }
                    }
                    __syncwarp();
                    for (int r = lane; r < total; r += 32) {
                        const int e = ring.list[r];
                        online_update_sample(m, s, kb, idx, tile_elem<DT>(tile, e), t0 + e, t0 + e, a.inv_tau, row_key);
                    }
                    __syncwarp();
                }
            }
            if (!compacted) {
#pragma unroll
            for (int j = 0; j < WPL; ++j) {
                // warp-uniform trip count (max popcount over the lanes); idle lanes feed -inf
                uint32_t b = bits[j];
                const int e0 = (j * 32 + lane) * 32;
                while (__any_sync(FULL, b != 0u)) {
                    const bool v = b != 0u;
                    const int e = e0 + (v ? (__ffs(b) - 1) : 0);
                    b &= b - 1u;
                    const float x = v ? tile_elem<DT>(tile, e) : -INFINITY;
                    if (SAMPLE)
                        online_update_sample(m, s, kb, idx, x, t0 + e, t0 + e, a.inv_tau, row_key);
                    else
                        online_update(m, s, idx, x, t0 + e);
                }
            }
            }
            }
            if (mt.flags & FLAG_LAST) {
                float rm = m, rs = s, rk = kb;
                int ri = idx;
                warp_combine_s<SAMPLE>(rm, rs, ri, rk);
                // SAMPLE: the tempered logit of the sampled token is re-read from the logits row
                auto sampled_y = [&](int pos) -> float {
                    if (!SAMPLE || rm == -INFINITY) return 0.0f;
                    const int tokid = gathered ? __ldg(a.dfa.tok + mt.csr_lo + pos) : pos;
                    const long long rr = gathered ? (long long)mt.tile : (long long)mt.pad;
                    const unsigned char* rowp = a.logits + rr * a.ld_bytes;
                    const float xv = (DT == DT_BF16)
                                         ? __uint_as_float(((uint32_t)__ldg(reinterpret_cast<const uint16_t*>(rowp) + tokid)) << 16)
                                         : __ldg(reinterpret_cast<const float*>(rowp) + tokid);
                    return __fmul_rn(xv, a.inv_tau);
                };
                if (np == 1) {
                    finalize_row(a, mt, rm, rs, ri, lane, gathered, SAMPLE, sampled_y(ri));
                } else {
                    // Publish from lane 1 (lane 0 is busy issuing copies): three self-validating
                    // words, then a RELAXED ticket -- no fence anywhere.  The last arriver merges.
                    int t = 0;
                    if (lane == 1) {
                        PartialSlot* ps = a.partials + ((long long)mt.slot * P + part);
                        st_relaxed_gpu_u64(&ps->m, tag | (unsigned)__float_as_int(rm));
                        st_relaxed_gpu_u64(&ps->s, tag | (unsigned)__float_as_int(rs));
                        st_relaxed_gpu_u64(&ps->idx, tag | (unsigned)ri);
                        if (SAMPLE) st_relaxed_gpu_u64(&ps->pad, tag | (unsigned)__float_as_int(rk));
                        t = atomicAdd(a.tickets + mt.slot, 1);
                    }
                    t = __shfl_sync(FULL, t, 1);
                    if (t == np - 1) {
                        if (lane == 1) a.tickets[mt.slot] = 0;
                        // The other units' words were stored before their tickets, but nothing
                        // orders them: poll until every tag is current (normally the first read).
                        const PartialSlot* base = a.partials + (long long)mt.slot * P;
                        // Merge in slot order whoever merges (bitwise reproducible): lane q%32 takes
                        // slot q; the own result (identical in every lane after the butterfly) stands
                        // in for slot `part`.
                        const float om = rm, os = rs, ok_ = rk;
                        const int oi = ri;
                        rm = -INFINITY;
                        rs = 0.0f;
                        rk = -INFINITY;
                        ri = 0x7FFFFFFF;
                        for (int q0 = 0; q0 < np; q0 += 32) {
                            const int q = q0 + lane;
                            const bool want = (q < np) && (q != part);
                            bool ok = !want;
                            unsigned long long wm = 0, ws = 0, wi = 0, wk = 0;
                            while (true) {
                                if (!ok) {
                                    wm = ld_relaxed_gpu_u64(&base[q].m);
                                    ws = ld_relaxed_gpu_u64(&base[q].s);
                                    wi = ld_relaxed_gpu_u64(&base[q].idx);
                                    ok = ((wm >> 32) == gen) && ((ws >> 32) == gen) && ((wi >> 32) == gen);
                                    if (SAMPLE) {
                                        wk = ld_relaxed_gpu_u64(&base[q].pad);
                                        ok = ok && ((wk >> 32) == gen);
                                    }
                                }
                                if (__all_sync(FULL, ok)) break;
                                __nanosleep(32);
                            }
                            if (SAMPLE) {
                                int dummy = 0;
                                if (want) {
                                    online_combine(rm, rs, dummy, __int_as_float((int)(unsigned)wm),
                                                   __int_as_float((int)(unsigned)ws), 0);
                                    sample_combine(rk, ri, __int_as_float((int)(unsigned)wk), (int)(unsigned)wi);
                                } else if (q == part) {
                                    online_combine(rm, rs, dummy, om, os, 0);
                                    sample_combine(rk, ri, ok_, oi);
                                }
                            } else if (want)
                                online_combine(rm, rs, ri, __int_as_float((int)(unsigned)wm),
                                               __int_as_float((int)(unsigned)ws), (int)(unsigned)wi);
                            else if (q == part)
                                online_combine(rm, rs, ri, om, os, oi);
                        }
                        warp_combine_s<SAMPLE>(rm, rs, ri, rk);
                        finalize_row(a, mt, rm, rs, ri, lane, gathered, SAMPLE, sampled_y(ri));
                    }
                }
            }
        }
        --in_flight;
        cons_stage = (cons_stage + 1 == STAGES) ? 0 : cons_stage + 1;
        cons_phase ^= (cons_stage == 0) ? 1u : 0u;
        __syncwarp();
        issue_one();
    }

    // ---------------- last CTA of the grid: reset the counters, then (decode loop) compact
    __shared__ int s_is_last;
    __syncthreads();
    if (threadIdx.x == 0) {
        const int d = atom_add_acq_rel_gpu(a.ctrs + 1, 1);
        s_is_last = (d == (int)gridDim.x - 1) ? 1 : 0;
        if (s_is_last) {
            a.ctrs[0] = 0;
            a.ctrs[1] = 0;
            a.ctrs[3] = (int)(gen + 1u);
        }
    }
    __syncthreads();
    if (s_is_last) {
        if (a.cmp_row_ids_out) {
            block_compact(a.done_out, a.row_map, a.state_new, n, a.cmp_row_ids_out, a.cmp_state_out, a.cmp_n_out);
            if (a.sat_ctr && threadIdx.x == 0 && __ldcg(a.sat_ctr) >= a.limit) *a.cmp_n_out = 0;
        } else {
            for (int i = threadIdx.x; i < n; i += blockDim.x) a.state[i] = __ldcg(a.state_new + i);
        }
    }
}

}  // namespace cd
