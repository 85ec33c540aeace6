// cd_step.cuh -- the fused constrained step (include/cd.h cd_step) and the
// persistent whole-loop kernel built from the same step body (cd_decode_loop).
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
//     of three 64-bit words, each carrying the launch generation in its upper half (8-byte stores
//     are single-copy atomic, so a word is either stale or complete), then takes a RELAXED
//     ticket.  The warp that draws the last ticket merges: it reads the other slots and re-reads
//     any word whose tag is not current yet (the writers issued those stores before their
//     tickets, so they are on their way; normally the first read succeeds).  A __threadfence
//     here cost 3.8 us per unit (profiles/r1b): it waits for the bulk copies the same warp still
//     has in flight.  Electing the merger in advance instead (the warp holding a row's last part
//     polls until the other parts are published: no atomic at all) was tried in round 2 and
//     dropped: a waiting warp streams nothing, and with 8 units per row an eighth of the warps
//     wait at any time -- c4 fell from 6.8 to 6.2 TB/s (profiles/r2_merge_election.md).
//   * The merging warp finds the chosen token's position in the state's CSR row WITHOUT searching:
//     position = number of allowed tokens below it = rank1k[state][t >> 10] (a per-state prefix
//     count of mask bits per 1024 tokens, built once with the automaton) + popcount of the mask
//     words of that block below t: one round trip instead of the 2-3 of a 128-ary search, then
//     next[] (accepting[next] rides in bit 31), the output writes and, in the decode loop, the
//     per-row history -- while the other warps keep streaming.
//   * step_kernel: one launch = one step.  The last CTA to finish resets the work counter, bumps
//     the generation and (per-step decode loops: callback / host-buffer forms) performs the
//     stable early-exit compaction.
//   * loop_kernel: one cooperative launch = the whole decode loop (cd_decode_loop).  148 CTAs stay
//     resident; between decoding steps they meet at a grid barrier (one arrival atomic per CTA,
//     the last arriver publishes the go word).  There is no compaction pass at all: the active set
//     is a bitmap over ORIGINAL row ids (three buffers in rotation: read / being built / being
//     cleared), finished rows simply do not set their bit for the next step, and "slot i" of a
//     step is the i-th set bit (rank/select on a shared-memory snapshot) -- which is exactly the
//     ascending-row-id order the stable compaction of a6 produces.  States live in two arrays
//     indexed by original row id (read k & 1, write (k + 1) & 1).  This removes, per decoding
//     step, a kernel launch + grid drain, the counter reset, the last-CTA compaction and the
//     active-count hand-off.
//   * Density-adaptive rows (GATHER instantiation): a row whose state has at most
//     `gather_max` transitions is not scanned at all -- its units walk pieces of the state's CSR
//     token list (coalesced) and gather exactly the allowed logits (one 32-byte sector each, 8
//     independent loads per lane in flight).  The running argmax is the CSR position, so the
//     transition needs no rank either.  Same outputs as the dense scan; dense and gathered rows
//     mix freely in one launch and share the merge machinery.
#pragma once
#include "cd_common.cuh"

namespace cd {

__device__ __forceinline__ unsigned long long global_timer_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}

constexpr int TPU_MAX_BYTES = 65536;  // at most 64 KiB of logits per unit
constexpr int UNITS_PER_WARP = 4;     // aim for >= this many units per warp when rows are few
constexpr int GATHER_UPW = 4;         // the same for gathered rows (pieces of the CSR token list)

constexpr int FLAG_FIRST = 1;   // first tile of its unit: reset the lane accumulators
constexpr int FLAG_LAST = 2;    // last tile of its unit: reduce and publish
constexpr int FLAG_ACCEPT = 4;  // pseudo tile of a slot whose state already accepts (no copy)
constexpr int FLAG_BADSTATE = 8;
constexpr int FLAG_GATHER = 16;  // pseudo tile of a gathered row piece (no copy)

constexpr int SAMPLE_LIST_CAP = 128;  // tiles with at most this many allowed elements are compacted (SAMPLE)

constexpr int GATHER_CHUNK = 256;  // a gathered row is split into pieces of >= this many transitions
constexpr int GATHER_UNROLL = 8;   // independent gathers per lane in flight

constexpr int LOOP_MAX_ROWS = 32768;     // persistent loop: rows per call (bitmap snapshot in shared memory)
constexpr int LOOP_PARAM_STEPS = 32;     // step pointers passed as kernel parameters up to this many steps
constexpr int LOOP_TRACE_STEPS = 256;    // per-step (timestamp, active rows) records kept for cd_loop_trace
constexpr unsigned long long LOOP_SPIN_TIMEOUT_NS = 4000000000ull;  // a barrier that waits longer aborts the loop
constexpr int FLOW_IDLE_LIMIT = 1 << 23;   // idle polls (>= 128 ns apart: > 1 s) after which a worker of flow_kernel gives up
constexpr int MERGE_SPIN_LIMIT = 1 << 24;  // polls (>= 32 ns apart) after which a merging warp gives up

// number of units a gathered row of `len` transitions is split into (P = units per row of the launch)
__host__ __device__ inline int gather_parts(int len, int P) {
    int np = (len + GATHER_CHUNK - 1) / GATHER_CHUNK;
    if (np < 1) np = 1;
    return np < P ? np : P;
}

// Result of one unit, readable without a fence: {gen:32 | payload:32} x 3 (+ the sampling key).
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
    int* token_out;    // per-slot outputs; all four may be NULL in the persistent loop
    float* logprob_out;
    float* lse_out;
    uint8_t* done_out;
    // scratch (per handle+stream)
    PartialSlot* partials;  // [units]
    int* tickets;           // [rows] arrivals per slot, zero between launches
    int* ctrs;              // [0] work counter, [1] finished CTAs, [2] error count, [3] generation
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
    // state with satisfying[s] != 0 are counted in *sat_ctr; once it reaches `limit` the active list is
    // emptied (every row still active is cancelled)
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
    int upw, tpu_max;  // unit sizing: target units per warp, most tiles per unit
    int idle_ns;       // flow_kernel: sleep between two looks at the groups' descriptors when nothing is published
};

// Persistent loop (loop_kernel): everything that outlives a step.
struct LoopArgs {
    const void* step_ptrs[LOOP_PARAM_STEPS];  // logits of step k, if max_steps <= LOOP_PARAM_STEPS ...
    const void* const* step_ptrs_dev;         // ... else a device array
    int B;
    uint32_t* alive[3];  // [nwords] active-row bitmaps in rotation: step k reads k % 3, builds (k + 1) % 3, clears (k + 2) % 3
    int* state2[2];      // [B] states by original row id: step k reads k & 1, writes (k + 1) & 1
    int* work;           // [max_steps] per-step work counters (zeroed by loop_init)
    int* bar;            // [0] arrivals, [1] go word: (steps completed) | stop << 30, [2] abort flag
    unsigned long long* trace_t;  // [LOOP_TRACE_STEPS + 1] globaltimer at the start of every step, then at exit
    int* trace_n;                 // [LOOP_TRACE_STEPS] active rows of every step, [LOOP_TRACE_STEPS] = steps run
    unsigned long long* phase;    // tuning builds (-DCD_TUNING): [LOOP_TRACE_STEPS][8] phase timestamps of every step
};

#ifdef CD_TUNING
#define CD_PHASE(L, k, i) do { if ((L).phase && (k) < LOOP_TRACE_STEPS) (L).phase[(k) * 8 + (i)] = global_timer_ns(); } while (0)
#define CD_PHASE_MAX(ptr) do { if (ptr) atomicMax(ptr, global_timer_ns()); } while (0)
#define CD_PHASE_MIN(ptr) do { if (ptr) atomicMax(ptr, ~global_timer_ns()); } while (0)  /* earliest = ~max(~t) */
#else
#define CD_PHASE(L, k, i) ((void)0)
#define CD_PHASE_MAX(ptr) ((void)0)
#define CD_PHASE_MIN(ptr) ((void)0)
#endif

// What changes from step to step (one launch of step_kernel, or one iteration of loop_kernel).
struct StepView {
    const unsigned char* logits;
    const int* state_cur;  // state of slot i (step_kernel) / of row r (loop_kernel)
    int* state_next;       // where finalize writes the next state (same indexing)
    int* work_ctr;
    unsigned gen;
    int n;
    int step;
    uint32_t* alive_next;  // loop_kernel: bitmap of the rows that stay active
    // loop_kernel: slot i = i-th set bit of the bitmap snapshot in shared memory
    const uint32_t* s_bits;
    const int* s_pref;  // exclusive prefix of the popcounts, [nwords + 1]
    int nwords;
    unsigned long long* ph_first_fin;  // tuning builds: earliest / latest row finalisation of the step
    unsigned long long* ph_last_fin;
    unsigned long long* ph_tile;  // tuning builds: [0] earliest (complemented), [1] latest first-tile arrival over the warps
};

struct __align__(16) TileMeta {
    int slot;
    int tile;   // tile index inside the row (gathered piece: unused)
    int flags;  // FLAG_* | part << 8
    int st;     // automaton state of the slot
    long long csr_lo;  // row_ptr[st]
    int csr_len;       // row_ptr[st + 1] - row_ptr[st]
    int lrow;          // row of the logits buffer
    // flow_kernel: the (group, step) this tile belongs to -- a warp's ring may hold tiles of several
    int step, n, tpu, grp;
};

constexpr int MODE_STEP = 0;  // step_kernel: one launch = one step
constexpr int MODE_LOOP = 1;  // loop_kernel: whole loop, grid barrier between steps (LIMIT loops)
constexpr int MODE_FLOW = 2;  // flow_kernel: whole loop, row groups advance independently (no barrier)

// flow_kernel (cd_decode_loop without a LIMIT): the rows are split into G groups of Bg consecutive
// original row ids, and every group is a decode loop of its own whose steps are published one by one:
//   desc[g]      {step:24 | n:24 | tpu:16} of the step whose units may be drawn now (DONE when the group is finished);
//                written with release by the warp that finalised the LAST row of the previous step of the group,
//                read with acquire by every warp before it draws a unit of that step
//   list[k&1]    [G*Bg] {row | state << 32}: the active rows of step k of each group, ascending row id (the stable
//                order of a6); listf[k&1] the running sum of log-probs of those rows (fp32 bits)
//   res / resf   [G*Bg] results of the running step by slot: {tag | done << 31 | next state}, {tag | new sum bits};
//                tag = launch generation + step, so a word is either stale or complete (as the partial slots)
//   fin[g]       rows finalised in the running step (relaxed counter: whoever brings it to n publishes the next step)
//   work         [G][max_steps] unit counters
// Nothing in it waits for a warp that is not running: units are only ever drawn by running warps.
struct FlowArgs {
    const void* step_ptrs[LOOP_PARAM_STEPS];
    const void* const* step_ptrs_dev;
    int B, G, Bg;
    unsigned long long* desc;
    unsigned long long* list[2];
    unsigned int* listf[2];
    unsigned long long* res;
    unsigned long long* resf;
    int* fin;
    int* work;
    long long pcap;  // partial slots per group
    unsigned long long* trace_t;  // [LOOP_TRACE_STEPS + 1] time at which the last group published step k; [steps] = exit
    int* trace_n;                 // [LOOP_TRACE_STEPS] active rows of step k over all groups; [LOOP_TRACE_STEPS] = steps run
};
constexpr unsigned long long FLOW_DONE = ~0ull;
constexpr int FLOW_MAX_GROUPS = 8;
__host__ __device__ inline unsigned long long flow_pack(int step, int n, int tpu) {
    return (unsigned long long)(unsigned)step | ((unsigned long long)(unsigned)n << 24) | ((unsigned long long)(unsigned)tpu << 48);
}

template <int STAGES, int TILE_BYTES>
struct __align__(128) WarpRing {
    unsigned char logits[STAGES][TILE_BYTES];
    unsigned char mask[STAGES][TILE_BYTES / 16];  // bf16: TILE_BYTES/2 tokens / 8; fp32 uses half
    TileMeta meta[STAGES];
    unsigned long long bar[STAGES];
    unsigned short list[SAMPLE_LIST_CAP];  // SAMPLE: positions of a tile's allowed elements, compacted
    int want[FLOW_MAX_GROUPS];             // flow_kernel: first step of each group this warp has not seen exhausted
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

// Position of token t inside the CSR row of state st = number of allowed tokens of st below t:
// the per-1024-token prefix count built with the automaton + the popcounts of the mask words of t's
// block below t (one word per lane).  Warp-uniform; one memory round trip.
__device__ __forceinline__ int mask_rank(const DfaDev& dfa, int st, int t, int lane) {
    const int blk = t >> 10, w = (t >> 5) & 31;
    const int wi = blk * 32 + lane;
    const uint32_t word = (wi < dfa.Wpad) ? __ldg(dfa.mask + (long long)st * dfa.Wpad + wi) : 0u;
    const int base = __ldg(dfa.rank1k + (long long)st * dfa.nblk + blk);
    int c = (lane < w) ? __popc(word) : ((lane == w) ? __popc(word & ((1u << (t & 31)) - 1u)) : 0);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(FULL, c, o);
    return base + c;
}

// flow_kernel: every row of step `step` of group `grp` is final -- build the group's next step.  Warp-
// cooperative.  The results of the step were stored by the rows' finalisers before their (relaxed) count,
// so they are on their way: poll until every tag is current.  Survivors keep their order (ascending row
// id: the stable compaction of a6).  The new step is published with a release store of its descriptor.
template <int WARPS>
__device__ __forceinline__ void flow_publish(const StepArgs& a, const FlowArgs& F, int grp, int step, int n, unsigned gen0,
                                             int tiles_per_row, int tpu_max, int lane) {
    const int kk = step + 1;
    const unsigned long long tag = (unsigned long long)(gen0 + (unsigned)step) << 32;
    const long long off = (long long)grp * F.Bg;
    const unsigned long long* cur = F.list[step & 1] + off;
    unsigned long long* nxt = F.list[kk & 1] + off;
    unsigned int* nxtf = F.listf[kk & 1] + off;
    int base = 0;
    constexpr int U = 4;  // chunks of 32 slots in flight
#pragma unroll 1
    for (int i0 = 0; i0 < n; i0 += 32 * U) {
        unsigned long long r[U], f[U], e[U];
#pragma unroll
        for (int q = 0; q < U; ++q) {
            const int i = i0 + q * 32 + lane;
            r[q] = f[q] = tag;
            e[q] = 0;
            if (i < n) {
                e[q] = ld_relaxed_gpu_u64(cur + i);
                int spins = 0;
                do {
                    r[q] = ld_relaxed_gpu_u64(F.res + off + i);
                    f[q] = ld_relaxed_gpu_u64(F.resf + off + i);
                } while (((r[q] ^ tag) >> 32 || (f[q] ^ tag) >> 32) && ++spins < MERGE_SPIN_LIMIT);
            }
        }
#pragma unroll
        for (int q = 0; q < U; ++q) {
            const int i = i0 + q * 32 + lane;
            const bool keep = (i < n) && (((unsigned)r[q] >> 31) == 0u) && !((r[q] ^ tag) >> 32);
            const unsigned b = __ballot_sync(FULL, keep);
            if (keep) {
                const int p = base + __popc(b & ((1u << lane) - 1u));
                nxt[p] = (e[q] & 0xFFFFFFFFull) | ((unsigned long long)((unsigned)r[q] & 0x7FFFFFFFu) << 32);
                nxtf[p] = (unsigned)f[q];
            }
            base += __popc(b);
        }
    }
    __syncwarp();
    if (lane == 0) {
        const bool stop = (base == 0) || (kk >= a.max_steps);
        F.fin[grp] = 0;
        if (stop) atomicMax(F.trace_n + LOOP_TRACE_STEPS, kk);  // steps run = the most any group ran
        if (kk <= LOOP_TRACE_STEPS) {
            if (kk < LOOP_TRACE_STEPS) atomicAdd(F.trace_n + kk, base);
            atomicMax(F.trace_t + kk, global_timer_ns());
        }
        const unsigned long long d =
            stop ? FLOW_DONE
                 // unit size as if all G groups had this many rows: the groups share the warps
                 : flow_pack(kk, base, tiles_per_unit((long long)base * F.G, tiles_per_row, (long long)gridDim.x * WARPS, tpu_max, a.upw));
        asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(F.desc + grp), "l"(d) : "memory");
    }
}

// Row finished: (m, s, idx) is the merged result of all its units.  Warp-uniform.
// `gathered`: idx is the position inside the state's CSR row instead of the token id.
// `sampled`: idx is the sampled token (position), ytok its tempered logit: logprob = (ytok - m) - log(sum).
// MODE_LOOP: per-row arrays are indexed by the original row id (mt.lrow); surviving rows set their bit in
// the next step's bitmap.  MODE_FLOW: the result goes to the group's result slots; returns true (in every
// lane) if this was the last row of the group's step (the caller then publishes the next step).
template <int MODE = MODE_STEP>
__device__ __forceinline__ bool finalize_row(const StepArgs& a, const StepView& sv, const FlowArgs* F, const TileMeta& mt,
                                             float m, float s, int idx, int lane, bool gathered, bool sampled = false,
                                             float ytok = 0.0f) {
    float lp, lse;
    int pos;
    long long csr_lo = mt.csr_lo;
    int csr_len = mt.csr_len;
    if (csr_len < 0) {  // dense-only kernels do not fetch the CSR bounds on the issue path: same round trip as the rank
        csr_lo = __ldg(a.dfa.row_ptr + mt.st);
        csr_len = (int)(__ldg(a.dfa.row_ptr + mt.st + 1) - csr_lo);
    }
    unsigned sum_prev_bits = 0;
    if (MODE == MODE_FLOW && lane == 0)  // the row's running sum travels with its list entry (same round trip as the rank)
        sum_prev_bits = __ldcg(F->listf[mt.step & 1] + (long long)mt.grp * F->Bg + mt.slot);
    if (m == -INFINITY) {  // every allowed logit is -inf: lowest allowed id (G6)
        lp = -INFINITY;
        lse = -INFINITY;
        pos = 0;
    } else {
        const float L = logf(s);
        lp = sampled ? (ytok - m) - L : -L;  // greedy: log p(t*) = -log(sum); never m - lse (cancellation)
        lse = m + L;
        pos = gathered ? idx : mask_rank(a.dfa, mt.st, idx, lane);
    }
    int last = 0;
    if (lane == 0) {
        const bool in_row = (pos >= 0) && (pos < csr_len);
        const long long j = csr_lo + pos;
        int token = in_row ? __ldg(a.dfa.tok + j) : -1;
        const int packed = in_row ? __ldg(a.dfa.next + j) : 0;  // next state | accepting << 31
        // the bitmask and the CSR describe the same set: the token found by rank must be the argmax
        const bool ok = in_row && (gathered || m == -INFINITY || token == idx);
        int ns = mt.st;
        uint8_t dn = 1;
        if (ok) {
            ns = packed & 0x7FFFFFFF;
            dn = (packed < 0) ? 1 : 0;
        } else {
            atomicAdd(a.ctrs + 2, 1);
            token = -1;
        }
        const int step = (MODE == MODE_FLOW) ? mt.step : sv.step;
        const int slot = (MODE == MODE_STEP) ? mt.slot : mt.lrow;
        CD_PHASE_MIN(sv.ph_first_fin);
        CD_PHASE_MAX(sv.ph_last_fin);
        if (MODE != MODE_FLOW) {
            sv.state_next[slot] = ns;
            if (a.token_out) a.token_out[slot] = token;
            if (a.logprob_out) a.logprob_out[slot] = lp;
            if (a.lse_out) a.lse_out[slot] = lse;
            if (a.done_out) a.done_out[slot] = dn;
        }
        if (MODE == MODE_LOOP && !dn) atomicOr(sv.alive_next + (slot >> 5), 1u << (slot & 31));
        if (a.hist_tokens) {  // decode loop: this slot's row, original id
            const long long rid = (MODE != MODE_STEP) ? (long long)mt.lrow : (a.row_map ? (long long)__ldg(a.row_map + slot) : slot);
            a.hist_tokens[rid * a.max_steps + step] = token;
            a.hist_len[rid] = step + 1;
            a.hist_final_state[rid] = ns;
            float sum;
            if (MODE == MODE_FLOW) sum = (step == 0 ? 0.0f : __uint_as_float(sum_prev_bits)) + lp;
            // (written by another SM one step ago in loop_kernel: read at the L2, never from a stale L1 line)
            else sum = __ldcg(a.hist_sum_logprob + rid) + lp;
            a.hist_sum_logprob[rid] = sum;
            a.hist_done[rid] = ok ? dn : (uint8_t)0;
            if (MODE != MODE_FLOW && a.sat_ctr && ok && dn && __ldg(a.satisfying + ns)) atomicAdd(a.sat_ctr, 1);
            if (MODE == MODE_FLOW) {
                const unsigned long long tag = (unsigned long long)(sv.gen + (unsigned)step) << 32;
                const long long o = (long long)mt.grp * F->Bg + mt.slot;
                st_relaxed_gpu_u64(F->res + o, tag | ((unsigned)ns & 0x7FFFFFFFu) | ((unsigned)dn << 31));
                st_relaxed_gpu_u64(F->resf + o, tag | __float_as_uint(sum));
                last = (atomicAdd(F->fin + mt.grp, 1) == mt.n - 1) ? 1 : 0;
            }
        }
    }
    if (MODE == MODE_FLOW) return __shfl_sync(FULL, last, 0) != 0;
    return false;
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

// Ring position of a warp: carried across the steps of the persistent loop (mbarrier phases go on).
struct RingPos {
    int iss_stage = 0;
    int cons_stage = 0;
    uint32_t cons_phase = 0;
};

// slot i of loop_kernel -> original row id: the i-th set bit of the snapshot (binary search over the
// per-word prefix counts, then find-nth-set inside the word).  Warp-uniform.
__device__ __forceinline__ int select_row(const StepView& sv, int i) {
    int lo = 0, hi = sv.nwords;  // invariant: s_pref[lo] <= i < s_pref[hi]
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (sv.s_pref[mid] <= i) lo = mid; else hi = mid;
    }
    const int r = i - sv.s_pref[lo];
    return lo * 32 + (int)__fns(sv.s_bits[lo], 0, r + 1);
}

// The step a unit belongs to: how its rows are split and where its shared state lives.
struct UnitCtx {
    int n, tpu, Pd, PG, P, total_units, step, grp;
    const unsigned char* logits;
    int* work;
    long long pbase;  // first partial slot
    int tbase;        // first ticket
};

template <int WARPS, int TILE_TOK, int TPU_MAX, bool GATHER>
__device__ __forceinline__ void unit_ctx_split(UnitCtx& c, const StepArgs& a, int n, int tpu) {
    const int total_warps = gridDim.x * WARPS;
    const int tiles_per_row = (a.dfa.V + TILE_TOK - 1) / TILE_TOK;
    c.n = n;
    c.tpu = tpu;
    c.Pd = (tiles_per_row + tpu - 1) / tpu;  // units per row of a dense scan
    // a gathered row is split only as far as needed to give every warp a few units
    c.PG = GATHER ? max(1, min(c.Pd, (total_warps * GATHER_UPW) / max(n, 1))) : c.Pd;
    // units per row of this step; if every state is gathered no unit is drawn in vain
    c.P = (GATHER && a.all_gather) ? c.PG : c.Pd;
    c.total_units = n * c.P;
}

// The streaming engine of a warp: issue + consume loops.
//   MODE_STEP / MODE_LOOP: one decoding step over the slots [0, sv.n); returns when the step's units are
//   exhausted and this warp's tiles are consumed.
//   MODE_FLOW: the whole loop; the warp draws units from whichever group has a published step with units
//   left (oldest step first) and returns when every group is finished.
template <int DT, int WARPS, int STAGES, int TILE_BYTES, bool GATHER, bool SAMPLE, int MODE>
__device__ __forceinline__ void step_body(const StepArgs& a, const StepView& sv, const FlowArgs* F,
                                          WarpRing<STAGES, TILE_BYTES>& ring, RingPos& rp, const int warp, const int lane) {
    constexpr int SZ = (DT == DT_BF16) ? 2 : 4;
    constexpr int TILE_TOK = TILE_BYTES / SZ;
    constexpr int MASK_BYTES = TILE_TOK / 8;
    constexpr int WPL = TILE_TOK / 1024;  // mask words per lane and tile
    constexpr int TPU_MAX = TPU_MAX_BYTES / TILE_BYTES;
    static_assert(WPL >= 1 && TILE_TOK % 1024 == 0, "tile must hold a multiple of 32 mask words");

    // ---------------- issue side (warp-uniform state)
    // MODE_STEP / MODE_LOOP: the first unit of a warp is its global warp id (no atomic on the start-up
    // chain); later units come from the work counter, which therefore starts at 0 = unit `total_warps`.
    // MODE_FLOW: every unit is drawn from its step's counter.
    const int total_warps = gridDim.x * WARPS;
    const int draw_base = (MODE == MODE_FLOW) ? 0 : total_warps;
    int next_u_l0 = blockIdx.x * WARPS + warp;  // prefetched unit id, valid in lane 0
    const int V = a.dfa.V;
    const int tiles_per_row = (V + TILE_TOK - 1) / TILE_TOK;
    const int tpu_max = min(TPU_MAX, a.tpu_max);
    UnitCtx cur{};
    bool have_step = false;   // MODE_FLOW: `cur` is a published step with units left (as far as this warp knows)
    bool all_done = false;    // MODE_FLOW: every group is finished
    if (MODE != MODE_FLOW) {
        unit_ctx_split<WARPS, TILE_TOK, TPU_MAX, GATHER>(cur, a, sv.n, tiles_per_unit(sv.n, tiles_per_row, total_warps, tpu_max, a.upw));
        cur.step = sv.step;
        cur.grp = 0;
        cur.logits = sv.logits;
        cur.work = sv.work_ctr;
        cur.pbase = 0;
        cur.tbase = 0;
        have_step = true;
    } else {
        if (lane < FLOW_MAX_GROUPS) ring.want[lane] = 0;
        __syncwarp();
    }
    const bool ragged_row = (V % TILE_TOK) != 0;
    const uint64_t pol_stream = l2_policy_evict_first();

    bool exhausted = false;
    int iss_tile = 0, iss_end = 0;
    int iss_slot = 0, iss_st = 0, iss_flags = 0, iss_len = 0, iss_row = 0;
    long long iss_lo = 0;
    const unsigned char* iss_src = nullptr;  // next logits tile of the current unit
    const unsigned char* iss_msk = nullptr;  // next mask piece
    int iss_stage = rp.iss_stage, in_flight = 0;

    // MODE_FLOW: look at the groups' descriptors (one per lane, acquire) and take the oldest published step
    // this warp has not seen exhausted; false if there is none right now
    auto acquire_step = [&]() -> bool {
        unsigned long long d = FLOW_DONE;
        if (lane < F->G) asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(d) : "l"(F->desc + lane) : "memory");
        const bool done_g = (lane >= F->G) || (d == FLOW_DONE);
        const int st_g = (int)(d & 0xFFFFFFull);
        const bool avail = !done_g && (st_g >= ring.want[lane & (FLOW_MAX_GROUPS - 1)]);
        if (__all_sync(FULL, done_g)) {
            all_done = true;
            return false;
        }
        int key = avail ? (st_g * FLOW_MAX_GROUPS + lane) : 0x7FFFFFFF;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) key = min(key, __shfl_xor_sync(FULL, key, o));
        if (key == 0x7FFFFFFF) return false;
        const int g = key & (FLOW_MAX_GROUPS - 1);
        d = __shfl_sync(FULL, d, g);
        const int step = (int)(d & 0xFFFFFFull), n = (int)((d >> 24) & 0xFFFFFFull), tpu = (int)(d >> 48);
        unit_ctx_split<WARPS, TILE_TOK, TPU_MAX, GATHER>(cur, a, n, tpu);
        cur.step = step;
        cur.grp = g;
        cur.logits = static_cast<const unsigned char*>(F->step_ptrs_dev ? F->step_ptrs_dev[step] : F->step_ptrs[step]);
        cur.work = F->work + (long long)g * a.max_steps + step;
        cur.pbase = (long long)g * F->pcap;
        cur.tbase = g * F->Bg;
        if (lane == 0) next_u_l0 = atomicAdd(cur.work, 1);
        have_step = true;
        return true;
    };

    // issues one tile (or pseudo tile); false if there is nothing to issue right now
    auto issue_one = [&]() -> bool {
        while (iss_tile >= iss_end) {  // next unit (units of a gathered row beyond its pieces are skipped)
            if (MODE == MODE_FLOW) {
                if (!have_step && !acquire_step()) return false;
            } else if (exhausted) {
                return false;
            }
            const int u = __shfl_sync(FULL, next_u_l0, 0);
            if (u >= cur.total_units) {
                if (MODE == MODE_FLOW) {  // this step has no units left: never look at it again
                    if (lane == 0) ring.want[cur.grp] = cur.step + 1;
                    __syncwarp();
                    have_step = false;
                    continue;
                }
                exhausted = true;
                return false;
            }
            if (lane == 0) next_u_l0 = draw_base + atomicAdd(cur.work, 1);
            iss_slot = u / cur.P;
            const int part = u - iss_slot * cur.P;
            long long rl;  // row of the logits buffer
            if (MODE == MODE_FLOW) {
                const unsigned long long e = ld_relaxed_gpu_u64(F->list[cur.step & 1] + (long long)cur.grp * F->Bg + iss_slot);
                rl = (long long)(unsigned)e;
                iss_st = (int)(e >> 32);
            } else if (MODE == MODE_LOOP) {
                rl = select_row(sv, iss_slot);
                // states are double-buffered by step parity: a unit drawn after its row was finalised
                // still sees the state the row was processed in
                iss_st = __ldcg(sv.state_cur + rl);
            } else {
                // state[] is not written while units are in flight (next states go to state_new[])
                iss_st = sv.state_cur[iss_slot];
                const long long r = a.row_map ? (long long)__ldg(a.row_map + iss_slot) : (long long)iss_slot;
                rl = a.logits_by_slot ? (long long)iss_slot : r;
            }
            iss_row = (int)rl;
            const bool bad = (iss_st < 0) || (iss_st >= a.dfa.S);
            const int sts = bad ? 0 : iss_st;
            // (the persistent loops never hold a row whose state accepts: such rows left the active set)
            const bool acc = (MODE == MODE_STEP) && !bad && (__ldg(a.dfa.accepting + sts) != 0);
            if (GATHER) {  // the CSR bounds decide between scan and gather
                iss_lo = __ldg(a.dfa.row_ptr + sts);
                iss_len = (int)(__ldg(a.dfa.row_ptr + sts + 1) - iss_lo);
            } else {  // dense only: nothing on the way to the first copy depends on them (finalize_row reads them)
                iss_lo = 0;
                iss_len = -1;
            }
            if (bad || acc) {
                if (lane == 0) {
                    ring.meta[iss_stage] = TileMeta{iss_slot, 0, (bad ? FLAG_BADSTATE : FLAG_ACCEPT) | (part << 8), iss_st, 0, 0,
                                                    iss_row, cur.step, cur.n, cur.tpu, cur.grp};
                    mbar_arrive(smem_u32(&ring.bar[iss_stage]));
                }
                iss_stage = (iss_stage + 1 == STAGES) ? 0 : iss_stage + 1;
                ++in_flight;
                iss_tile = iss_end = 0;
                return true;
            }
            if (GATHER && iss_len <= a.gather_max) {
                if (part >= gather_parts(iss_len, cur.PG)) continue;
                if (lane == 0) {
                    ring.meta[iss_stage] = TileMeta{iss_slot, 0, FLAG_GATHER | FLAG_LAST | (part << 8), iss_st, iss_lo, iss_len,
                                                    iss_row, cur.step, cur.n, cur.tpu, cur.grp};
                    mbar_arrive(smem_u32(&ring.bar[iss_stage]));
                }
                iss_stage = (iss_stage + 1 == STAGES) ? 0 : iss_stage + 1;
                ++in_flight;
                iss_tile = iss_end = 0;
                return true;
            }
            iss_tile = part * cur.tpu;
            iss_end = min(iss_tile + cur.tpu, tiles_per_row);
            iss_src = cur.logits + rl * a.ld_bytes + (long long)iss_tile * TILE_BYTES;
            iss_msk = reinterpret_cast<const unsigned char*>(a.dfa.mask + (long long)iss_st * a.dfa.Wpad) +
                      (long long)iss_tile * MASK_BYTES;
            iss_flags = (part << 8) | FLAG_FIRST;
        }
        const uint32_t bar = smem_u32(&ring.bar[iss_stage]);
        const uint32_t dst = smem_u32(ring.logits[iss_stage]);
        const uint32_t mdst = smem_u32(ring.mask[iss_stage]);
        const int fl = iss_flags | ((iss_tile + 1 == iss_end) ? FLAG_LAST : 0);
        const TileMeta meta{iss_slot, iss_tile, fl, iss_st, iss_lo, iss_len, iss_row, cur.step, cur.n, cur.tpu, cur.grp};
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
                ring.meta[iss_stage] = meta;
                mbar_arrive_expect_tx(bar, bulk + mbytes);
                if (bulk) bulk_g2s_hint(dst, iss_src, bulk, bar, pol_stream);
                bulk_g2s(mdst, iss_msk, mbytes, bar);
            }
        } else if (lane == 0) {
            ring.meta[iss_stage] = meta;
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
        return true;
    };

    // ---------------- consume side
    float m = -INFINITY, s = 0.0f, kb = -INFINITY;  // kb: best perturbed key (SAMPLE); idx then is its token
    int idx = 0x7FFFFFFF;
    int cons_stage = rp.cons_stage;
    uint32_t cons_phase = rp.cons_phase;
#ifdef CD_TUNING
    bool first_tile = true;
#endif
    int idle_polls = 0;

#pragma unroll 1
    for (;;) {
        while (in_flight < STAGES && issue_one()) {
        }
        if (in_flight == 0) {
            if (MODE != MODE_FLOW || all_done) break;
            __nanosleep(a.idle_ns);  // nothing published right now: some group is between two steps
            if (++idle_polls > FLOW_IDLE_LIMIT) {  // never on a healthy run: fail the call, do not hang
                if (lane == 0) atomicAdd(a.ctrs + 2, 1);
                break;
            }
            continue;
        }
        idle_polls = 0;
        mbar_wait(smem_u32(&ring.bar[cons_stage]), cons_phase);
        __syncwarp();
#ifdef CD_TUNING
        if (first_tile && sv.ph_tile && lane == 0) {
            atomicMax(sv.ph_tile, ~global_timer_ns());
            atomicMax(sv.ph_tile + 1, global_timer_ns());
        }
        first_tile = false;
#endif
        const TileMeta mt = ring.meta[cons_stage];
        const int part = mt.flags >> 8;
        // the step this tile belongs to (MODE_FLOW: whatever the ring holds; else the step of this call)
        UnitCtx cc = cur;
        if (MODE == MODE_FLOW) {
            unit_ctx_split<WARPS, TILE_TOK, TPU_MAX, GATHER>(cc, a, mt.n, mt.tpu);
            cc.step = mt.step;
            cc.grp = mt.grp;
            cc.logits = static_cast<const unsigned char*>(F->step_ptrs_dev ? F->step_ptrs_dev[mt.step] : F->step_ptrs[mt.step]);
            cc.pbase = (long long)mt.grp * F->pcap;
            cc.tbase = mt.grp * F->Bg;
        }
        const unsigned gen = sv.gen + ((MODE == MODE_FLOW) ? (unsigned)cc.step : 0u);  // tag of the partial slots
        const unsigned long long tag = (unsigned long long)gen << 32;
        const int rng_step = a.rng_step_base + cc.step;
        // original row id of the slot: names the history row and seeds the sampling noise
        auto orig_row = [&]() -> uint32_t {
            return (MODE != MODE_STEP) ? (uint32_t)mt.lrow : (uint32_t)(a.row_map ? __ldg(a.row_map + mt.slot) : mt.slot);
        };
        bool publish = false;  // MODE_FLOW: this warp finalised the last row of (cc.grp, cc.step)

        if (mt.flags & (FLAG_ACCEPT | FLAG_BADSTATE)) {
            // accepted rows never advance; a state outside [0, S) is reported done
            if (part == 0) {
                int last = 0;
                if (lane == 0) {
                    const int slot = (MODE == MODE_STEP) ? mt.slot : mt.lrow;
                    if (MODE != MODE_FLOW) {
                        sv.state_next[slot] = mt.st;
                        if (a.token_out) a.token_out[slot] = -1;
                        if (a.logprob_out) a.logprob_out[slot] = 0.0f;
                        if (a.lse_out) a.lse_out[slot] = 0.0f;
                        if (a.done_out) a.done_out[slot] = 1;
                    }
                    if (mt.flags & FLAG_BADSTATE) {
                        atomicAdd(a.ctrs + 2, 1);
                        if (a.hist_tokens) {  // the row leaves the loop here, undone, in the state it has
                            const long long rid = orig_row();
                            a.hist_final_state[rid] = mt.st;
                            a.hist_done[rid] = 0;
                        }
                    }
                    if (MODE == MODE_FLOW) {  // the row leaves its group
                        const long long o = (long long)mt.grp * F->Bg + mt.slot;
                        st_relaxed_gpu_u64(F->res + o, tag | 0x80000000u);
                        st_relaxed_gpu_u64(F->resf + o, tag);
                        last = (atomicAdd(F->fin + mt.grp, 1) == mt.n - 1) ? 1 : 0;
                    }
                }
                if (MODE == MODE_FLOW) publish = __shfl_sync(FULL, last, 0) != 0;
            }
        } else {
            const bool gathered = GATHER && (mt.flags & FLAG_GATHER);
            const int np = gathered ? gather_parts(mt.csr_len, cc.PG) : cc.P;  // units this row was split into
            if (gathered) {
                // piece [j0, j1) of the state's CSR row: tokens read coalesced, their logits gathered
                // with GATHER_UNROLL independent loads per lane; idx = position in the CSR row, which
                // ascends with the token id, so "replace on strictly greater" keeps the lowest id
                m = -INFINITY;
                s = 0.0f;
                kb = -INFINITY;
                idx = 0x7FFFFFFF;
                const uint32_t row_key = SAMPLE ? rng_row_key(a.seed_lo, a.seed_hi, orig_row(), (uint32_t)rng_step) : 0u;
                const int j0 = (int)(((long long)mt.csr_len * part) / np);
                const int j1 = (int)(((long long)mt.csr_len * (part + 1)) / np);
                const int* tk = a.dfa.tok + mt.csr_lo;
                const unsigned char* rowp = cc.logits + (long long)mt.lrow * a.ld_bytes;
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
                const uint32_t row_key = SAMPLE ? rng_row_key(a.seed_lo, a.seed_hi, orig_row(), (uint32_t)rng_step) : 0u;
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
                    const unsigned char* rowp = cc.logits + (long long)mt.lrow * a.ld_bytes;
                    const float xv = (DT == DT_BF16)
                                         ? __uint_as_float(((uint32_t)__ldg(reinterpret_cast<const uint16_t*>(rowp) + tokid)) << 16)
                                         : __ldg(reinterpret_cast<const float*>(rowp) + tokid);
                    return __fmul_rn(xv, a.inv_tau);
                };
                if (np == 1) {
                    publish = finalize_row<MODE>(a, sv, F, mt, rm, rs, ri, lane, gathered, SAMPLE, sampled_y(ri));
                } else {
                    // Publish from lane 1 (lane 0 is busy issuing copies): self-validating words,
                    // then a RELAXED ticket -- no fence anywhere.  The last arriver merges.
                    int t = 0;
                    if (lane == 1) {
                        PartialSlot* ps = a.partials + (cc.pbase + (long long)mt.slot * cc.P + part);
                        st_relaxed_gpu_u64(&ps->m, tag | (unsigned)__float_as_int(rm));
                        st_relaxed_gpu_u64(&ps->s, tag | (unsigned)__float_as_int(rs));
                        st_relaxed_gpu_u64(&ps->idx, tag | (unsigned)ri);
                        if (SAMPLE) st_relaxed_gpu_u64(&ps->pad, tag | (unsigned)__float_as_int(rk));
                        t = atomicAdd(a.tickets + cc.tbase + mt.slot, 1);
                    }
                    t = __shfl_sync(FULL, t, 1);
                    if (t == np - 1) {
                        if (lane == 1) a.tickets[cc.tbase + mt.slot] = 0;
                        // The other units' words were stored before their tickets, but nothing orders
                        // them: poll until every tag is current (normally the first read).
                        const PartialSlot* base = a.partials + (cc.pbase + (long long)mt.slot * cc.P);
                        // Merge in slot order whoever merges (bitwise reproducible): lane q % 32 takes
                        // slot q; the own result (identical in every lane after the butterfly) stands in
                        // for slot `part`.
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
                            int spins = 0;
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
                                if (++spins > MERGE_SPIN_LIMIT) {  // never on a healthy run: fail the call, do not hang
                                    if (lane == 0) atomicAdd(a.ctrs + 2, 1);
                                    break;
                                }
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
                        publish = finalize_row<MODE>(a, sv, F, mt, rm, rs, ri, lane, gathered, SAMPLE, sampled_y(ri));
                    }
                }
            }
        }
        if (MODE == MODE_FLOW && publish)
            flow_publish<WARPS>(a, *F, cc.grp, cc.step, cc.n, sv.gen, tiles_per_row, tpu_max, lane);
        --in_flight;
        cons_stage = (cons_stage + 1 == STAGES) ? 0 : cons_stage + 1;
        cons_phase ^= (cons_stage == 0) ? 1u : 0u;
        __syncwarp();
    }
    rp.iss_stage = iss_stage;
    rp.cons_stage = cons_stage;
    rp.cons_phase = cons_phase;
}

// ------------------------------------------------------------------ one launch = one step (cd_step)
template <int DT, int WARPS, int STAGES, int TILE_BYTES, bool GATHER, bool SAMPLE = false>
__global__ void __launch_bounds__(WARPS * 32, 1) step_kernel(const StepArgs a) {
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

    StepView sv{};
    sv.logits = a.logits;
    sv.state_cur = a.state;
    sv.state_next = a.state_new;
    sv.work_ctr = a.ctrs + 0;
    sv.gen = (unsigned)__ldcg(a.ctrs + 3);
    sv.n = a.n_dev ? __ldcg(a.n_dev) : a.n;
    sv.step = a.step;
    RingPos rp;
    step_body<DT, WARPS, STAGES, TILE_BYTES, GATHER, SAMPLE, MODE_STEP>(a, sv, nullptr, ring, rp, warp, lane);

    // ---------------- last CTA of the grid: reset the counters, then (decode loop) compact
    __shared__ int s_is_last;
    __syncthreads();
    if (threadIdx.x == 0) {
        const int d = atom_add_acq_rel_gpu(a.ctrs + 1, 1);
        s_is_last = (d == (int)gridDim.x - 1) ? 1 : 0;
        if (s_is_last) {
            a.ctrs[0] = 0;
            a.ctrs[1] = 0;
            a.ctrs[3] = (int)(sv.gen + 1u);
        }
    }
    __syncthreads();
    if (s_is_last) {
        if (a.cmp_row_ids_out) {
            block_compact(a.done_out, a.row_map, a.state_new, sv.n, a.cmp_row_ids_out, a.cmp_state_out, a.cmp_n_out);
            if (a.sat_ctr && threadIdx.x == 0 && __ldcg(a.sat_ctr) >= a.limit) *a.cmp_n_out = 0;
        } else {
            for (int i = threadIdx.x; i < sv.n; i += blockDim.x) a.state[i] = __ldcg(a.state_new + i);
        }
    }
}

// ------------------------------------------------------------------ one launch = the whole loop
__device__ __forceinline__ int ld_acquire_gpu_s32(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu_s32(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Grid barrier after decoding step k (k1 = k + 1 barriers completed once everybody is through).  The
// last arriver has observed every finalisation of the step (acq_rel arrival chain), so it decides the
// LIMIT stop there, once, for the whole grid, and publishes it with the go word.  Returns the go word's
// flags: bit 0 = stop (LIMIT reached or abort).
__device__ __forceinline__ int loop_barrier(const LoopArgs& L, int k1, const int* sat_ctr, int limit) {
    __shared__ int s_go;
    __syncthreads();
    if (threadIdx.x == 0) {
        const int old = atom_add_acq_rel_gpu(L.bar + 0, 1);
        if (old == k1 * (int)gridDim.x - 1) {
            const int stop = (sat_ctr && __ldcg(sat_ctr) >= limit) ? 1 : 0;
            st_release_gpu_s32(L.bar + 1, k1 | (stop << 30));
        }
        int v;
        const unsigned long long t0 = global_timer_ns();
        while (((v = ld_acquire_gpu_s32(L.bar + 1)) & 0x3FFFFFFF) < k1) {
            if (ld_acquire_gpu_s32(L.bar + 2) != 0) { v = k1 | (1 << 30); break; }
            if (global_timer_ns() - t0 > LOOP_SPIN_TIMEOUT_NS) {  // never on a healthy device: fail, do not hang
                atomicExch(L.bar + 2, 1);
                v = k1 | (1 << 30);
                break;
            }
        }
        s_go = v;
    }
    __syncthreads();
    return (s_go >> 30) & 1;
}

template <int DT, int WARPS, int STAGES, int TILE_BYTES, bool GATHER, bool SAMPLE = false>
__global__ void __launch_bounds__(WARPS * 32, 1) loop_kernel(const StepArgs a, const LoopArgs L) {
    using Ring = WarpRing<STAGES, TILE_BYTES>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    Ring& ring = reinterpret_cast<Ring*>(smem_raw)[warp];
    const int nwords = (L.B + 31) >> 5;
    uint32_t* s_bits = reinterpret_cast<uint32_t*>(smem_raw + sizeof(Ring) * WARPS);
    int* s_pref = reinterpret_cast<int*>(s_bits + nwords);  // [nwords + 1]

    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) mbar_init(smem_u32(&ring.bar[s]), 1);
        fence_mbar_init();
    }
    __syncwarp();

    const unsigned gen0 = (unsigned)__ldcg(a.ctrs + 3);
    RingPos rp;
    int k = 0;
#pragma unroll 1
    for (; k < a.max_steps; ++k) {
        // ---- snapshot of the active-row bitmap -> shared memory, per-word prefix counts, n
        const uint32_t* cur = L.alive[k % 3];
        for (int w = threadIdx.x; w < nwords; w += WARPS * 32) s_bits[w] = __ldcg(cur + w);
        __syncthreads();
        if (warp == 0) {
            int carry = 0;
            for (int w0 = 0; w0 < nwords; w0 += 32) {
                const int w = w0 + lane;
                const int c = (w < nwords) ? __popc(s_bits[w]) : 0;
                int inc = c;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int up = __shfl_up_sync(FULL, inc, o);
                    if (lane >= o) inc += up;
                }
                if (w < nwords) s_pref[w] = carry + inc - c;
                carry += __shfl_sync(FULL, inc, 31);
            }
            if (lane == 0) s_pref[nwords] = carry;
        }
        __syncthreads();
        const int n = s_pref[nwords];
        if (blockIdx.x == 0 && threadIdx.x == 0 && k < LOOP_TRACE_STEPS) {
            L.trace_t[k] = global_timer_ns();
            L.trace_n[k] = n;
        }
        if (blockIdx.x == 0 && threadIdx.x == 0) CD_PHASE(L, k, 0);  // snapshot done
        if (n == 0) break;  // every CTA reads the same bitmap: uniform across the grid
        // the bitmap read two steps from now was last read one step ago: clear it (nobody touches it
        // before the next barrier)
        if (blockIdx.x == 0) {
            uint32_t* clr = L.alive[(k + 2) % 3];
            for (int w = threadIdx.x; w < nwords; w += WARPS * 32) clr[w] = 0u;
        }

        StepView sv{};
        sv.logits = static_cast<const unsigned char*>(L.step_ptrs_dev ? L.step_ptrs_dev[k] : L.step_ptrs[k]);
        sv.state_cur = L.state2[k & 1];
        sv.state_next = L.state2[(k + 1) & 1];
        sv.work_ctr = L.work + k;
        sv.gen = gen0 + (unsigned)k;
        sv.n = n;
        sv.step = k;
        sv.alive_next = L.alive[(k + 1) % 3];
        sv.s_bits = s_bits;
        sv.s_pref = s_pref;
        sv.nwords = nwords;
#ifdef CD_TUNING
        if (L.phase && k < LOOP_TRACE_STEPS) {
            sv.ph_first_fin = L.phase + k * 8 + 2;
            sv.ph_last_fin = L.phase + k * 8 + 3;
            sv.ph_tile = L.phase + k * 8 + 5;
        }
#endif
        step_body<DT, WARPS, STAGES, TILE_BYTES, GATHER, SAMPLE, MODE_LOOP>(a, sv, nullptr, ring, rp, warp, lane);
        if (blockIdx.x == 0 && threadIdx.x == 0) CD_PHASE(L, k, 1);  // CTA 0 / warp 0 ran out of work
#ifdef CD_TUNING
        __syncthreads();
        if (threadIdx.x == 0 && L.phase && k < LOOP_TRACE_STEPS) atomicMax(L.phase + k * 8 + 4, global_timer_ns());  // last CTA at the barrier
#endif

        if (loop_barrier(L, k + 1, a.sat_ctr, a.limit)) {
            ++k;
            break;
        }
    }
    // ---------------- last CTA to leave: generation for the next launch, trace end
    if (threadIdx.x == 0) {
        const int d = atom_add_acq_rel_gpu(a.ctrs + 1, 1);
        if (d == (int)gridDim.x - 1) {
            a.ctrs[1] = 0;
            a.ctrs[3] = (int)(gen0 + (unsigned)a.max_steps + 1u);
            const int kk = k < LOOP_TRACE_STEPS ? k : LOOP_TRACE_STEPS;
            L.trace_t[kk] = global_timer_ns();
            L.trace_n[LOOP_TRACE_STEPS] = k;
        }
    }
}

// ------------------------------------------------------------------ one launch = the whole loop, no barrier
// cd_decode_loop without a LIMIT.  Every warp is an independent worker: it draws units from whichever row
// group has a published step with units left (oldest step first, so the groups stay staggered: while one
// group is between two steps -- last rows being merged, transition looked up, next step published -- the
// others keep the memory system busy), and returns when every group is finished.  There is no block-wide
// or grid-wide synchronisation after the ring set-up, and no warp ever waits for a warp that is not
// running, so the launch needs no co-residency guarantee.
template <int DT, int WARPS, int STAGES, int TILE_BYTES, bool GATHER, bool SAMPLE = false>
__global__ void __launch_bounds__(WARPS * 32, 1) flow_kernel(const StepArgs a, const FlowArgs F) {
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
    const unsigned gen0 = (unsigned)__ldcg(a.ctrs + 3);
    if (blockIdx.x == 0 && threadIdx.x == 0) atomicMax(F.trace_t + 0, global_timer_ns());
    StepView sv{};
    sv.gen = gen0;
    RingPos rp;
    step_body<DT, WARPS, STAGES, TILE_BYTES, GATHER, SAMPLE, MODE_FLOW>(a, sv, &F, ring, rp, warp, lane);
    // ---------------- last CTA to leave: generation for the next launch
    __syncthreads();
    if (threadIdx.x == 0) {
        const int d = atom_add_acq_rel_gpu(a.ctrs + 1, 1);
        if (d == (int)gridDim.x - 1) {
            a.ctrs[1] = 0;
            a.ctrs[3] = (int)(gen0 + (unsigned)a.max_steps + 1u);
        }
    }
}

}  // namespace cd
