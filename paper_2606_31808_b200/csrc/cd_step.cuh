// cd_step.cuh -- the fused constrained step (include/cd.h cd_step) and the two
// persistent whole-loop kernels built from the same step body (cd_decode_loop).
//
// Design (B200-first; the paper gives no kernel):
//   * The step is one streaming pass over the logits, so it is HBM-bound: the job is to keep
//     enough bytes in flight and to waste no issue slots.  Every WARP owns a private ring of
//     STAGES shared-memory slots that it fills itself with 1-D bulk async copies (TMA engine,
//     cp.async.bulk -> SASS UBLKCP) completing on per-slot mbarriers: a logits tile and the
//     matching piece of the state's allowed-token bitmask land together.  No register staging,
//     no block-wide barriers in the streaming phase, WARPS*STAGES*TILE_BYTES in flight per SM.
//   * Work unit = (active slot, range of whole chunks of the row).  Units are handed out by one global
//     atomic counter (dynamic balance across the 148 SMs; the two dies do not run at the same speed).
//   * Per tile: a sparse tile (the normal case) is compacted across the warp -- one scan of the per-lane
//     popcounts, the allowed positions in a small shared list -- and every lane evaluates its fair share of
//     the ALLOWED elements only, updating an online (max, sum-exp, argmax) triple; a dense tile walks the set
//     bits of the lane's mask words as independent chains.  Warp reductions go through the redux unit.
//   * CANONICAL CHUNKS: a row is cut into chunks (a function of V and the logits type only); a chunk's result
//     is a fixed function of its elements, the row's a fixed fold of its chunks' results.  How a launch cuts
//     rows into units therefore never changes a bit of logprob / lse (see MAX_CHUNKS below).
//   * Chunk results travel through HBM without any fence: three 64-bit words, each carrying the launch
//     generation in its upper half (8-byte stores are single-copy atomic, so a word is either stale or
//     complete); a unit then adds its number of chunks to the row's RELAXED ticket and whoever completes the
//     row merges, re-reading any word whose tag is not current yet (the writers issued those stores before
//     their tickets, so they are on their way; normally the first read succeeds).  A __threadfence here cost
//     3.8 us per unit (profiles/r1b): it waits for the bulk copies the same warp still has in flight.
//   * The merging warp finds the chosen token's position in the state's CSR row WITHOUT searching:
//     position = number of allowed tokens below it = rank1k[state][t >> 10] (a per-state prefix
//     count of mask bits per 1024 tokens, built once with the automaton) + popcount of the mask
//     words of that block below t: one round trip instead of the 2-3 of a 128-ary search, then
//     next[] (accepting[next] rides in bit 31), the output writes and, in the decode loop, the
//     per-row history -- while the other warps keep streaming.
//   * step_kernel: one launch = one step (cd_step; the callback / host-buffer loops).  The last CTA to finish
//     resets the work counter, bumps the generation and (loops) performs the stable early-exit compaction.
//   * loop_kernel: one cooperative launch = the whole decode loop in lock-step (LIMIT loops).  148 CTAs stay
//     resident; between decoding steps they meet at a grid barrier (one arrival atomic per CTA,
//     the last arriver publishes the go word).  There is no compaction pass at all: the active set
//     is a bitmap over ORIGINAL row ids (three buffers in rotation: read / being built / being
//     cleared), finished rows simply do not set their bit for the next step, and "slot i" of a
//     step is the i-th set bit (rank/select on a shared-memory snapshot) -- which is exactly the
//     ascending-row-id order the stable compaction of a6 produces.
//   * flow_kernel: one plain launch = the whole decode loop with NO barrier (cd_decode_loop): every row
//     advances through its steps on its own; the warp that finalises a row's step publishes the next one as
//     entries of a queue ring, cut into more units the idler the machine is (see FlowArgs).
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

// Canonical arithmetic (the same bits whatever the launch): a row is cut into CHUNKS -- chunk_tiles()
// consecutive tiles each, at most MAX_CHUNKS per row, a function of V and the logits type only.  The result
// of a chunk is the warp combination of the 32 lane chains over its elements (ascending token id per lane); the
// result of a row is: lane l folds the chunk results l, l + 32 in ascending order, then the same warp
// combination.  A UNIT (what one warp draws) is a range of whole chunks, so how a row is cut into units -- which
// depends on the number of active rows, on the kernel and, in flow_kernel, on how busy the machine is when the
// row's step is published -- never changes a bit of the result: logprob / lse of a row are the same from cd_step
// on one row and from a 4096-row decode loop.  A gathered row has its own canonical pieces (gather_piece()).
constexpr int MAX_CHUNKS = 64;
#ifndef CD_CHUNK_TILES
#define CD_CHUNK_TILES 1
#endif
constexpr int CHUNK_TILES = CD_CHUNK_TILES;

constexpr int FLAG_FIRST = 1;   // first tile of its chunk: reset the lane accumulators
constexpr int FLAG_LAST = 2;    // last tile of its chunk: reduce and publish the chunk's result
constexpr int FLAG_ACCEPT = 4;  // pseudo tile of a slot whose state already accepts (no copy)
constexpr int FLAG_BADSTATE = 8;
constexpr int FLAG_GATHER = 16;  // pseudo tile of a gathered row's unit (no copy)
constexpr int FLAG_UEND = 32;    // last tile of its unit: take the ticket
// TileMeta.flags: bits 8-15 = chunk index (dense tile) / part (pseudo tiles), bits 16-23 = chunks of the unit
// (dense tile) / parts the gathered row is split into

constexpr int TILE_LIST_CAP = 128;  // tiles with at most this many allowed elements are compacted across the warp

constexpr int GATHER_CHUNK = 256;  // a gathered row is cut into pieces of >= this many transitions
constexpr int GATHER_UNROLL = 8;   // independent gathers per lane in flight

constexpr int LOOP_MAX_ROWS = 32768;     // persistent loop: rows per call (bitmap snapshot in shared memory)
constexpr int LOOP_PARAM_STEPS = 32;     // step pointers passed as kernel parameters up to this many steps
constexpr int LOOP_TRACE_STEPS = 256;    // per-step (timestamp, active rows) records kept for cd_loop_trace
constexpr unsigned long long LOOP_SPIN_TIMEOUT_NS = 4000000000ull;  // a barrier that waits longer aborts the loop
constexpr int FLOW_IDLE_LIMIT = 1 << 23;   // idle polls (>= 128 ns apart: > 1 s) after which a worker of flow_kernel gives up
constexpr int MERGE_SPIN_LIMIT = 1 << 24;  // polls (>= 32 ns apart) after which a merging warp gives up
// loop_kernel's barrier words, one 128-byte line each (the go word and the abort flag are polled by every CTA while
// the arrivals are counted with atomics)
constexpr int LB_ARRIVE = 0, LB_GO = 32, LB_ABORT = 64, LB_INTS = 96;
constexpr int FLOW_ENTRY_WORDS = 8;        // 64-byte queue entries (5 words used)
// flow_kernel's counters, one 128-byte line each (the stop word is polled by every idle warp: kept away from the
// lines the unit draws and the publications hit with atomics)
constexpr int FQ_DRAWN = 0, FQ_PUBLISHED = 32, FQ_FINISHED = 64, FQ_ERRORS = 96, FQ_LAUNCHES = 97, FQ_STOP = 128;
// the stop word exists in FQ_STOP_COPIES lines (warp w reads copy w % FQ_STOP_COPIES): every idle warp can look at it
// on every poll without 1,700 warps reading one line
constexpr int FQ_STOP_COPIES = 64;
constexpr int FQ_INTS = FQ_STOP + 32 * FQ_STOP_COPIES;

// tiles per chunk / chunks per row of a row of `tiles_per_row` tiles
__host__ __device__ inline int chunk_tiles(int tiles_per_row) {
    const int c = (tiles_per_row + MAX_CHUNKS - 1) / MAX_CHUNKS;
    return c < CHUNK_TILES ? CHUNK_TILES : c;
}
__host__ __device__ inline int row_chunks(int tiles_per_row) {
    const int ct = chunk_tiles(tiles_per_row);
    return (tiles_per_row + ct - 1) / ct;
}
// canonical pieces of a gathered row of `len` transitions: piece size (a multiple of 32) and count (<= MAX_CHUNKS)
__host__ __device__ inline int gather_piece(int len) {
    int p = (len + MAX_CHUNKS - 1) / MAX_CHUNKS;
    p = (p + 31) & ~31;
    return p < GATHER_CHUNK ? GATHER_CHUNK : p;
}
__host__ __device__ inline int gather_pieces(int len) {
    const int g = gather_piece(len);
    const int n = (len + g - 1) / g;
    return n < 1 ? 1 : n;
}
// units a dense row is cut into when n rows are active (host mirrors this: cd_api.cu flow_units0)
__host__ __device__ inline int units_per_row(long long n, int tiles_per_row, long long total_warps, int tpu_max,
                                             int upw = UNITS_PER_WARP) {
    const int ct = chunk_tiles(tiles_per_row);
    const int tc = (tiles_per_row + ct - 1) / ct;
    long long cpu = (n * tc + total_warps * upw - 1) / (total_warps * upw);  // chunks per unit
    int cpu_max = tpu_max / ct;
    if (cpu_max < 1) cpu_max = 1;
    if (cpu < 1) cpu = 1;
    if (cpu > cpu_max) cpu = cpu_max;
    return (int)((tc + cpu - 1) / cpu);
}

// Result of one chunk, readable without a fence: {gen:32 | payload:32} x 3 (+ the sampling key).
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
    PartialSlot* partials;  // [rows][pstride]
    int pstride;            // chunk-result slots per row: the most chunks / gathered pieces a row of this automaton can have
    int* tickets;           // [2 * rows] chunks arrived per slot (flow_kernel: per row and step parity), zero between uses
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
    int force_p;       // tuning builds: > 0 = units per dense row, whatever the number of rows
    int idle_ns;       // flow_kernel: sleep between two looks at an unpublished queue entry
};

// Persistent loop (loop_kernel): everything that outlives a step.
struct LoopArgs {
    const void* step_ptrs[LOOP_PARAM_STEPS];  // logits of step k, if max_steps <= LOOP_PARAM_STEPS ...
    const void* const* step_ptrs_dev;         // ... else a device array
    int B;
    uint32_t* alive[3];  // [nwords] active-row bitmaps in rotation: step k reads k % 3, builds (k + 1) % 3, clears (k + 2) % 3
    int* state2[2];      // [B] states by original row id: step k reads k & 1, writes (k + 1) & 1
    int* work;           // [max_steps] per-step work counters (zeroed by loop_init)
    int* bar;            // [LB_INTS]: arrivals, go word: (steps completed) | stop << 30, abort flag -- one 128-byte line each
    unsigned long long* trace_t;  // [LOOP_TRACE_STEPS + 1] globaltimer at the start of every step, then at exit
    int* trace_n;                 // [LOOP_TRACE_STEPS] active rows of every step, [LOOP_TRACE_STEPS] = steps run
    unsigned long long* phase;    // tuning builds (-DCD_TUNING): [LOOP_TRACE_STEPS][8] phase timestamps of every step
};

#ifdef CD_TUNING
#define CD_PHASE(L, k, i) do { if ((L).phase && (k) < LOOP_TRACE_STEPS) (L).phase[(k) * 8 + (i)] = global_timer_ns(); } while (0)
#define CD_PHASE_MAX(ptr) do { if (ptr) atomicMax(ptr, global_timer_ns()); } while (0)
#define CD_PHASE_MIN(ptr) do { if (ptr) atomicMax(ptr, ~global_timer_ns()); } while (0)  /* earliest = ~max(~t) */
// flow_kernel, per row step (record row * max_steps + step): [0] published [1] ~first / [2] last unit resolved
// [3] last unit streamed [4] merger drew the last ticket [5] merger has the chunk results [6] transition read
// [7] ~first tile landed
#define CD_DBG_MAX(F, rec, i) do { if ((F) && (F)->dbg && (rec) < (F)->dbg_cap) atomicMax((F)->dbg + (long long)(rec) * 16 + (i), global_timer_ns()); } while (0)
#define CD_DBG_MIN(F, rec, i) do { if ((F) && (F)->dbg && (rec) < (F)->dbg_cap) atomicMax((F)->dbg + (long long)(rec) * 16 + (i), ~global_timer_ns()); } while (0)
// [8..15] largest SM-clock cycle counts: [8] copy issue -> landed [9] landed -> elements done [10] chunk result + publish
// [11] ticket -> merged [12] merged -> published
#define CD_DBG_CYC(F, rec, i, v) do { if ((F) && (F)->dbg && (rec) < (F)->dbg_cap) atomicMax((F)->dbg + (long long)(rec) * 16 + (i), (unsigned long long)(v)); } while (0)
#define CD_CLOCK() ((unsigned)clock64())
#else
#define CD_DBG_CYC(F, rec, i, v) ((void)0)
#define CD_CLOCK() 0u
#define CD_DBG_MAX(F, rec, i) ((void)0)
#define CD_DBG_MIN(F, rec, i) ((void)0)
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
    unsigned long long* trace_t;  // flow_kernel: the trace buffers of this launch
    int* trace_n;
    unsigned long long* ph_first_fin;  // tuning builds: earliest / latest row finalisation of the step
    unsigned long long* ph_last_fin;
    unsigned long long* ph_tile;  // tuning builds: [0] earliest (complemented), [1] latest first-tile arrival over the warps
};

struct __align__(16) TileMeta {
    int slot;
    int tile;   // tile index inside the row (pseudo tiles: unused)
    int flags;  // FLAG_* | chunk or part << 8 | chunks of the unit or parts of the row << 16
    int st;     // automaton state of the slot
    long long csr_lo;  // row_ptr[st]
    int csr_len;       // row_ptr[st + 1] - row_ptr[st]
    int lrow;          // row of the logits buffer
    // flow_kernel: the step this tile belongs to (a warp's ring may hold tiles of several) and the row's running
    // sum of log-probs before it (fp32 bits; travels with the row)
    int step;
    unsigned sumbits;
    int pad[2];
};

constexpr int MODE_STEP = 0;  // step_kernel: one launch = one step
constexpr int MODE_LOOP = 1;  // loop_kernel: whole loop, grid barrier between steps (LIMIT loops)
constexpr int MODE_FLOW = 2;  // flow_kernel: whole loop, every row advances on its own (no barrier)

// flow_kernel (cd_decode_loop without a LIMIT): rows are independent, so nothing makes row r
// wait at step k for the other rows.  What is scheduled is a UNIT = a range of chunks of one decoding step of
// one row, drawn in order from one counter (q[0]):
//   units 0 .. B * P0 - 1 are implicit: unit u = part u % P0 of P0 of (row u / P0, start state, step 0, sum 0)
//     -- nothing is read to start them;
//   unit B * P0 + e is entry e of the queue `task` (a ring of cap = 2^cap_log2 entries of 64 bytes; entry e
//     lives at e % cap).  Five self-validating words {tag : 32 | payload : 32}, tag = launch generation + e / cap:
//       [0] original row id  [1] automaton state  [2] running sum of log-probs (fp32 bits)  [3] step
//       [4] part | parts << 8 (the unit is part `part` of `parts` of the row's chunks)
//     written (relaxed, no fence) by the warp that finalised the row's previous step, at the indices it reserved
//     with one atomicAdd on q[1]; a word is either stale (older tag) or complete.  A row has at most MAX_CHUNKS
//     entries that are reserved and not read yet, and it reserves the entries of its next step only after every
//     unit of this one has been read, so with cap >= B * MAX_CHUNKS at most cap entries are UNREAD at any time.
//     That bounds their number, not the span of indices they cover: a warp holds the id of its next unit while it
//     finishes the current one, and if the other rows meanwhile publish a full ring of entries (cap is 2 * B * chunks,
//     at least 1024: possible only for a handful of rows running hundreds of steps past a stalled warp) the slot is
//     rewritten with a later tag before that warp reads it.  The tag check turns this into a reader that never
//     sees its tag -- the idle timeout ends the loop with CD_ERR_INTERNAL -- never into a wrong result.
//   HOW MANY units a row's next step is cut into is decided when it is published, from how busy the machine is
//   (entries published minus units drawn): the row's full set of chunks when warps are waiting for work -- the few
//   rows of a long tail then spread over the whole machine and a step costs one chunk's latency --, down to
//   64 KiB units when every warp already has work queued.  The canonical arithmetic (see MAX_CHUNKS) makes the
//   result independent of that decision, so results stay bitwise reproducible.
//   A warp whose next unit is not published yet keeps consuming what its ring holds, then polls the entry (and
//   the stop word).  Units taken from the counter are only ever drawn by running warps and every published unit is
//   drawn before any later one.  The FIRST unit of a warp is not drawn: it is the warp's global id (see step_body),
//   so the rows of step 0 are started only once every CTA of the launch has run -- the launch needs all its CTAs to
//   get an SM eventually.  A kernel that ends frees them; ANOTHER flow loop does not end before its own CTAs all
//   ran, so two of them on one device could hold each other up until the idle timeout.  The host orders these
//   launches across the streams of a process (cd_api.cu FlowOrder); loops of different processes are not covered.
//   q[2] counts the rows that left the loop (accepted, truncated at max_steps, failed); whoever brings it to B
//   stores the launch generation into q[3], the stop word.  The last CTA to leave resets q[0..2], reports the
//   error count q[4] to host_status (pinned, mapped host memory: no copy after the loop) and counts the launch
//   in q[5], whose parity selects the trace buffers (the other pair is cleared for the next launch).
// No set-up kernel: a row's outputs (len, final state, sum, done, the -1 padding of its token history) are
// written by the warp that finalises its last step.
struct FlowArgs {
    const void* step_ptrs[LOOP_PARAM_STEPS];
    const void* const* step_ptrs_dev;
    int B;
    int start;  // start state
    unsigned long long* task;  // [cap][FLOW_ENTRY_WORDS]
    unsigned cap_mask;         // cap - 1
    int cap_log2;
    // units a published row step is cut into, by how busy the machine is: backlog (units published and not drawn
    // yet; negative = warps waiting) >= th[i] -> np_lvl[i], below th[2] -> np_lvl[3] (every chunk a unit)
    int np_lvl[4];
    int th[3];
    int* q;                    // [0] units drawn [1] entries reserved [2] rows finished [3] stop word [4] errors [5] launches
    unsigned long long* trace_t[2];  // [LOOP_TRACE_STEPS + 1] latest publication of a task of step k; [steps] = exit
    int* trace_n[2];                 // [LOOP_TRACE_STEPS] rows that ran step k; [LOOP_TRACE_STEPS] = steps run
    int* host_status;                // [0] errors of the loops since the host last cleared it
    unsigned long long* dbg;         // tuning builds: [dbg_cap][8] phase timestamps per row step (see CD_DBG_*)
    int dbg_cap;
};

template <int STAGES, int TILE_BYTES>
struct __align__(128) WarpRing {
    unsigned char logits[STAGES][TILE_BYTES];
    unsigned char mask[STAGES][TILE_BYTES / 16];  // bf16: TILE_BYTES/2 tokens / 8; fp32 uses half
    TileMeta meta[STAGES];
    unsigned long long bar[STAGES];
    unsigned short list[TILE_LIST_CAP];  // positions of a sparse tile's allowed elements, compacted
};

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

// flow_kernel: row `rid` leaves the loop after `steps` steps -- its outputs are final.  Warp-cooperative: the
// rest of its token history is padded with -1 (no set-up kernel did).  Whoever brings the count of finished rows
// to B stores the stop word.
__device__ __forceinline__ void flow_row_leaves(const StepArgs& a, const StepView& sv, const FlowArgs& F, long long rid,
                                                int steps, int state, float sum, uint8_t done, int lane) {
    for (int k = steps + lane; k < a.max_steps; k += 32) a.hist_tokens[rid * a.max_steps + k] = -1;
    if (lane == 0) {
        a.hist_len[rid] = steps;
        a.hist_final_state[rid] = state;
        a.hist_sum_logprob[rid] = sum;
        a.hist_done[rid] = done;
        atomicMax(sv.trace_n + LOOP_TRACE_STEPS, steps);  // steps run = the most any row ran
    }
    int last = 0;
    if (lane == 0) last = (atomicAdd(F.q + FQ_FINISHED, 1) == F.B - 1) ? 1 : 0;
    if (__shfl_sync(FULL, last, 0))  // the loop is over: every copy of the stop word
        for (int i = lane; i < FQ_STOP_COPIES; i += 32) atomicExch(F.q + FQ_STOP + 32 * i, (int)sv.gen);
}

// Row finished: (m, s, idx) is the merged result of all its chunks.  Warp-uniform.
// `gathered`: idx is the position inside the state's CSR row instead of the token id.
// `sampled`: idx is the sampled token (position), ytok its tempered logit: logprob = (ytok - m) - log(sum).
// MODE_LOOP: per-row arrays are indexed by the original row id (mt.lrow); surviving rows set their bit in
// the next step's bitmap.  MODE_FLOW: a surviving row's next step is published as new queue entries (q0 / q1 =
// units drawn / entries reserved as read a moment ago: how busy the machine is); a row that is done, truncated
// or failed leaves the loop.
template <int MODE = MODE_STEP>
__device__ __forceinline__ void finalize_row(const StepArgs& a, const StepView& sv, const FlowArgs* F, const TileMeta& mt,
                                             float m, float s, int idx, int lane, bool gathered, bool sampled = false,
                                             float ytok = 0.0f, int q0 = 0, int q1 = 0, long long units0 = 0) {
    float lp, lse;
    int pos;
    long long csr_lo = mt.csr_lo;
    int csr_len = mt.csr_len;
    if (csr_len < 0) {  // dense-only kernels do not fetch the CSR bounds on the issue path: same round trip as the rank
        csr_lo = __ldg(a.dfa.row_ptr + mt.st);
        csr_len = (int)(__ldg(a.dfa.row_ptr + mt.st + 1) - csr_lo);
    }
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
    int leave = 0, ns = mt.st, cont = 0;
    uint8_t dn = 1;
    float sum = 0.0f;
    const int step = (MODE == MODE_FLOW) ? mt.step : sv.step;
    if (lane == 0) {
        const bool in_row = (pos >= 0) && (pos < csr_len);
        const long long j = csr_lo + pos;
        int token = in_row ? __ldg(a.dfa.tok + j) : -1;
        const int packed = in_row ? __ldg(a.dfa.next + j) : 0;  // next state | accepting << 31
        // the bitmask and the CSR describe the same set: the token found by rank must be the argmax
        const bool ok = in_row && (gathered || m == -INFINITY || token == idx);
        if (ok) {
            ns = packed & 0x7FFFFFFF;
            dn = (packed < 0) ? 1 : 0;
        } else {
            atomicAdd(MODE == MODE_FLOW ? F->q + FQ_ERRORS : a.ctrs + 2, 1);
            token = -1;
        }
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
        if (MODE == MODE_FLOW) {
            const long long rid = mt.lrow;
            a.hist_tokens[rid * a.max_steps + step] = token;
            sum = __uint_as_float(mt.sumbits) + lp;  // step 0: 0.0f + lp
            CD_DBG_MAX(F, rid * a.max_steps + step, 6);
            if (!dn && step + 1 < a.max_steps) {
                cont = 1;
            } else {
                leave = 1;
                if (!ok) dn = 0;  // a failed row is reported undone
            }
        } else if (a.hist_tokens) {  // decode loop: this slot's row, original id
            const long long rid = (MODE != MODE_STEP) ? (long long)mt.lrow : (a.row_map ? (long long)__ldg(a.row_map + slot) : slot);
            a.hist_tokens[rid * a.max_steps + step] = token;
            a.hist_len[rid] = step + 1;
            a.hist_final_state[rid] = ns;
            // (written by another SM one step ago in loop_kernel: read at the L2, never from a stale L1 line)
            a.hist_sum_logprob[rid] = __ldcg(a.hist_sum_logprob + rid) + lp;
            a.hist_done[rid] = ok ? dn : (uint8_t)0;
            if (a.sat_ctr && ok && dn && __ldg(a.satisfying + ns)) atomicAdd(a.sat_ctr, 1);
        }
    }
    if (MODE == MODE_FLOW) {
        cont = __shfl_sync(FULL, cont, 0);
        ns = __shfl_sync(FULL, ns, 0);
        sum = __shfl_sync(FULL, sum, 0);
        if (cont) {
            // how many units for the row's next step: all its chunks if warps are waiting for work, 64 KiB units
            // if every warp has work queued (backlog = units published and not drawn yet)
            const long long backlog = units0 + q1 - q0;
            const int np = (backlog >= F->th[0]) ? F->np_lvl[0] : ((backlog >= F->th[1]) ? F->np_lvl[1] : ((backlog >= F->th[2]) ? F->np_lvl[2] : F->np_lvl[3]));
            unsigned e0 = 0;
            if (lane == 0) e0 = (unsigned)atomicAdd(F->q + FQ_PUBLISHED, np);
            e0 = __shfl_sync(FULL, e0, 0);
            const unsigned w0 = (unsigned)mt.lrow, w1 = (unsigned)ns, w2 = __float_as_uint(sum), w3 = (unsigned)(step + 1);
            for (int i = lane; i < np; i += 32) {
                const unsigned e = e0 + (unsigned)i;
                unsigned long long* ent = F->task + (size_t)(e & F->cap_mask) * FLOW_ENTRY_WORDS;
                const unsigned long long tag = (unsigned long long)(sv.gen + (e >> F->cap_log2)) << 32;
                st_relaxed_gpu_u64(ent + 0, tag | w0);
                st_relaxed_gpu_u64(ent + 1, tag | w1);
                st_relaxed_gpu_u64(ent + 2, tag | w2);
                st_relaxed_gpu_u64(ent + 3, tag | w3);
                st_relaxed_gpu_u64(ent + 4, tag | (unsigned)(i | (np << 8)));
            }
            if (lane == 0) {
                CD_DBG_MAX(F, (long long)mt.lrow * a.max_steps + step + 1, 0);
                if (step + 1 < LOOP_TRACE_STEPS) {
                    atomicAdd(sv.trace_n + step + 1, 1);
                    atomicMax(sv.trace_t + step + 1, global_timer_ns());
                }
            }
        }
        leave = __shfl_sync(FULL, leave, 0);
        if (leave)
            flow_row_leaves(a, sv, *F, mt.lrow, step + 1, ns, sum, (uint8_t)__shfl_sync(FULL, (int)dn, 0), lane);
    }
}

template <bool SAMPLE>
__device__ __forceinline__ void warp_combine_s(float& m, float& s, int& idx, float& kb) {
    if constexpr (!SAMPLE) {
        warp_combine_redux(m, s, idx);
    } else {
        int dummy = 0x7FFFFFFF;
        warp_combine_redux(m, s, dummy);
        warp_argmax_redux(kb, idx);
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

// How the rows of a step (MODE_STEP / MODE_LOOP) or the implicit first step (MODE_FLOW) are cut into units.
struct UnitCtx {
    int n, Pd, PG, P, total_units, step;
    const unsigned char* logits;
    int* work;
};

template <int WARPS, bool GATHER>
__device__ __forceinline__ void unit_ctx_split(UnitCtx& c, const StepArgs& a, int n, int tiles_per_row, int tpu_max) {
    const int total_warps = gridDim.x * WARPS;
    c.n = n;
    c.Pd = units_per_row(n, tiles_per_row, total_warps, tpu_max, a.upw);  // units per row of a dense scan
    if (a.force_p > 0) c.Pd = min(a.force_p, row_chunks(tiles_per_row));
    // a gathered row is split only as far as needed to give every warp a few units
    c.PG = GATHER ? max(1, min(c.Pd, (total_warps * GATHER_UPW) / max(n, 1))) : c.Pd;
    // units per row of this step; if every state is gathered no unit is drawn in vain
    c.P = (GATHER && a.all_gather) ? c.PG : c.Pd;
    c.total_units = n * c.P;
}

// The streaming engine of a warp: issue + consume loops.
//   MODE_STEP / MODE_LOOP: one decoding step over the slots [0, sv.n); returns when the step's units are
//   exhausted and this warp's tiles are consumed.
//   MODE_FLOW: the whole loop; the warp draws units (see FlowArgs) and returns when every row has left the loop.
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
    // The first unit of a warp is its global warp id (no atomic on the start-up chain: 1,776 warps drawing from one
    // address at once); later units come from the work counter, which therefore starts at 0 = unit `total_warps`.
    const int total_warps = gridDim.x * WARPS;
    const int draw_base = total_warps;
    int next_u_l0 = blockIdx.x * WARPS + warp;  // prefetched unit id, valid in lane 0
    const int V = a.dfa.V;
    const int tiles_per_row = (V + TILE_TOK - 1) / TILE_TOK;
    const int CT = chunk_tiles(tiles_per_row);              // tiles per chunk
    const int Tc = (tiles_per_row + CT - 1) / CT;           // chunks per row
    const int tpu_max = min(TPU_MAX, a.tpu_max);
    UnitCtx cur{};
    bool all_done = false;      // MODE_FLOW: every row has left the loop
    bool poll_pending = false;  // MODE_FLOW: poll_w / poll_stop hold the loads issued for the unit in next_u_l0
    unsigned long long poll_w = 0;
    int poll_stop = 0;
    long long units0 = 0;  // MODE_FLOW: implicit units (the first step of every row)
    if (MODE != MODE_FLOW) {
        unit_ctx_split<WARPS, GATHER>(cur, a, sv.n, tiles_per_row, tpu_max);
        cur.step = sv.step;
        cur.logits = sv.logits;
        cur.work = sv.work_ctr;
    } else {
        unit_ctx_split<WARPS, GATHER>(cur, a, F->B, tiles_per_row, tpu_max);
        units0 = (long long)F->B * cur.P;
        cur.work = F->q + FQ_DRAWN;
    }
    const bool ragged_row = (V % TILE_TOK) != 0;
    const uint64_t pol_stream = l2_policy_evict_first();

    bool exhausted = false;
    int iss_tile = 0, iss_end = 0, iss_in_chunk = 0, iss_nch = 0;
    int iss_slot = 0, iss_st = 0, iss_len = 0, iss_row = 0, iss_step = 0;
    unsigned iss_sum = 0u;
    long long iss_lo = 0;
    const unsigned char* iss_src = nullptr;  // next logits tile of the current unit
    const unsigned char* iss_msk = nullptr;  // next mask piece
    int iss_stage = rp.iss_stage, in_flight = 0;

    // issues one tile (or pseudo tile); false if there is nothing to issue right now
    auto issue_one = [&]() -> bool {
        while (iss_tile >= iss_end) {  // next unit (units of a gathered row beyond its pieces are skipped)
            if (MODE == MODE_FLOW ? all_done : exhausted) return false;
            const int u = __shfl_sync(FULL, next_u_l0, 0);
            long long rl;  // row of the logits buffer
            int part, np;  // this unit is part `part` of `np` of its row
            if (MODE == MODE_FLOW) {
                iss_step = 0;
                iss_sum = 0u;
                if (u < units0) {  // implicit unit: row u / P takes step 0 from the start state
                    const int q = u / cur.P;
                    part = u - q * cur.P;
                    np = cur.P;
                    rl = q;
                    iss_st = F->start;
                } else {
                    // lanes 0-4: the entry's words; lane 5: the stop word (one round trip for both).  The loads are
                    // issued here and looked at on the NEXT call: meanwhile the warp consumes a tile (or sleeps),
                    // so a poll never stalls the consume side.
                    const unsigned e = (unsigned)((long long)u - units0);
                    const unsigned expect = sv.gen + (e >> F->cap_log2);
                    const bool fresh = poll_pending && (unsigned)(poll_w >> 32) == expect;
                    const bool ready = poll_pending && __all_sync(FULL, lane >= 5 || fresh);
                    if (!ready) {  // not published (yet)
                        if (poll_pending && (unsigned)__shfl_sync(FULL, poll_stop, 5) == sv.gen) all_done = true;
                        poll_w = 0;
                        if (lane < 5) poll_w = ld_relaxed_gpu_u64(F->task + (size_t)(e & F->cap_mask) * FLOW_ENTRY_WORDS + lane);
                        if (lane == 5) poll_stop = ld_relaxed_gpu_s32(F->q + FQ_STOP + 32 * ((blockIdx.x * WARPS + warp) % FQ_STOP_COPIES));
                        poll_pending = true;
                        return false;
                    }
                    poll_pending = false;
                    const unsigned long long w = poll_w;
                    rl = (long long)(unsigned)__shfl_sync(FULL, w, 0);
                    iss_st = (int)(unsigned)__shfl_sync(FULL, w, 1);
                    iss_sum = (unsigned)__shfl_sync(FULL, w, 2);
                    iss_step = (int)(unsigned)__shfl_sync(FULL, w, 3);
                    const unsigned pn = (unsigned)__shfl_sync(FULL, w, 4);
                    part = (int)(pn & 0xFFu);
                    np = (int)((pn >> 8) & 0xFFu);
                }
                // (drawing the next unit only when the last tile of this one is issued -- so that the warps that have
                // waited longest, not the ones that just took work, hold the next ids -- was tried: the draw and the
                // poll then sit in front of every unit's first copy; c4 lost 2 %, the tail gained nothing)
                if (lane == 0) next_u_l0 = draw_base + atomicAdd(cur.work, 1);
                if (lane == 0) {
                    CD_DBG_MIN(F, rl * a.max_steps + iss_step, 1);
                    CD_DBG_MAX(F, rl * a.max_steps + iss_step, 2);
                }
                iss_slot = (int)rl;
                cur.step = iss_step;
                cur.logits = static_cast<const unsigned char*>(F->step_ptrs_dev ? F->step_ptrs_dev[iss_step] : F->step_ptrs[iss_step]);
            } else {
                if (u >= cur.total_units) {
                    exhausted = true;
                    return false;
                }
                if (lane == 0) next_u_l0 = draw_base + atomicAdd(cur.work, 1);
                iss_slot = u / cur.P;
                part = u - iss_slot * cur.P;
                np = cur.P;
                if (MODE == MODE_LOOP) {
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
                                                    iss_row, iss_step, iss_sum, {0, 0}};
                    mbar_arrive(smem_u32(&ring.bar[iss_stage]));
                }
                iss_stage = (iss_stage + 1 == STAGES) ? 0 : iss_stage + 1;
                ++in_flight;
                iss_tile = iss_end = 0;
                return true;
            }
            if (GATHER && iss_len <= a.gather_max) {
                // a gathered row is cut into at most as many units as it has canonical pieces
                const int parts = min(gather_pieces(iss_len), (MODE == MODE_FLOW) ? np : cur.PG);
                if (part >= parts) continue;
                if (lane == 0) {
                    ring.meta[iss_stage] = TileMeta{iss_slot, 0, FLAG_GATHER | (part << 8) | (parts << 16), iss_st, iss_lo, iss_len,
                                                    iss_row, iss_step, iss_sum, {0, 0}};
                    mbar_arrive(smem_u32(&ring.bar[iss_stage]));
                }
                iss_stage = (iss_stage + 1 == STAGES) ? 0 : iss_stage + 1;
                ++in_flight;
                iss_tile = iss_end = 0;
                return true;
            }
            // dense: chunks [Tc * part / np, Tc * (part + 1) / np)
            const int c0 = (int)(((long long)Tc * part) / np), c1 = (int)(((long long)Tc * (part + 1)) / np);
            iss_nch = c1 - c0;
            iss_tile = c0 * CT;
            iss_end = min(c1 * CT, tiles_per_row);
            iss_in_chunk = 0;
            iss_src = cur.logits + rl * a.ld_bytes + (long long)iss_tile * TILE_BYTES;
            iss_msk = reinterpret_cast<const unsigned char*>(a.dfa.mask + (long long)iss_st * a.dfa.Wpad) +
                      (long long)iss_tile * MASK_BYTES;
        }
        const uint32_t bar = smem_u32(&ring.bar[iss_stage]);
        const uint32_t dst = smem_u32(ring.logits[iss_stage]);
        const uint32_t mdst = smem_u32(ring.mask[iss_stage]);
        const bool chunk_ends = (iss_in_chunk + 1 == CT) || (iss_tile + 1 == tiles_per_row);
        const int chunk = (CT == 1) ? iss_tile : iss_tile / CT;
        const int fl = ((iss_in_chunk == 0) ? FLAG_FIRST : 0) | (chunk_ends ? FLAG_LAST : 0) |
                       ((iss_tile + 1 == iss_end) ? FLAG_UEND : 0) | (chunk << 8) | (iss_nch << 16);
        const TileMeta meta{iss_slot, iss_tile, fl, iss_st, iss_lo, iss_len, iss_row, iss_step, iss_sum, {0, (int)CD_CLOCK()}};
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
        iss_in_chunk = chunk_ends ? 0 : iss_in_chunk + 1;
        iss_src += TILE_BYTES;
        iss_msk += MASK_BYTES;
        ++iss_tile;
        ++in_flight;
        iss_stage = (iss_stage + 1 == STAGES) ? 0 : iss_stage + 1;
        return true;
    };

    // ---------------- consume side
    // NC independent chains per lane (greedy: one per mask word of a tile, so that a lone warp is not bound by
    // the latency of one dependent chain of online updates; sampling keeps one): chain j of lane l sees the
    // elements of word j * 32 + l of every tile of the chunk, in ascending token id
    constexpr int NC = SAMPLE ? 1 : WPL;
    float am[NC], as[NC];
    int ai[NC];
    float kb = -INFINITY;  // best perturbed key (SAMPLE); ai[0] then is its token
    bool many_chains = false;  // warp-uniform: a chain other than chain 0 was fed since the last reset
    auto reset_chains = [&]() {
        many_chains = false;
#pragma unroll
        for (int j = 0; j < NC; ++j) {
            am[j] = -INFINITY;
            as[j] = 0.0f;
            ai[j] = 0x7FFFFFFF;
        }
        kb = -INFINITY;
    };
    // the lane's chains -> one (m, s, idx) (pairwise tree; equal maxima keep the lower token id), then the warp
    auto chunk_result = [&](float& rm, float& rs, int& ri, float& rk) {
        if (NC > 1 && many_chains) {  // (combining with an untouched chain changes nothing: skipping it is exact)
#pragma unroll
            for (int w = 1; w < NC; w <<= 1) {
#pragma unroll
                for (int j = 0; j + w < NC; j += 2 * w) online_combine(am[j], as[j], ai[j], am[j + w], as[j + w], ai[j + w]);
            }
        }
        rm = am[0];
        rs = as[0];
        ri = ai[0];
        rk = kb;
        warp_combine_s<SAMPLE>(rm, rs, ri, rk);
    };
    reset_chains();
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
            __nanosleep(a.idle_ns);  // this warp's next unit is not published yet
            if (++idle_polls > FLOW_IDLE_LIMIT) {  // never on a healthy run: fail the call, do not hang
                if (lane == 0) atomicAdd(F->q + FQ_ERRORS, 1);
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
        const int fpart = (mt.flags >> 8) & 0xFF;   // chunk index (dense) / part (pseudo tiles)
        const int fcnt = (mt.flags >> 16) & 0xFF;   // chunks of the unit (dense) / parts of the row (gathered)
        // the step this tile belongs to (MODE_FLOW: whatever the ring holds; else the step of this call)
        const int tstep = (MODE == MODE_FLOW) ? mt.step : cur.step;
        const unsigned char* tlogits =
            (MODE == MODE_FLOW) ? static_cast<const unsigned char*>(F->step_ptrs_dev ? F->step_ptrs_dev[mt.step] : F->step_ptrs[mt.step])
                                : cur.logits;
        const unsigned gen = sv.gen + ((MODE == MODE_FLOW) ? (unsigned)tstep : 0u);  // tag of the chunk results
        const unsigned long long tag = (unsigned long long)gen << 32;
        const int rng_step = a.rng_step_base + tstep;
        const long long dbg_rec = (MODE == MODE_FLOW) ? (long long)mt.lrow * a.max_steps + tstep : 0;
        (void)dbg_rec;
        // original row id of the slot: names the history row and seeds the sampling noise
        auto orig_row = [&]() -> uint32_t {
            return (MODE != MODE_STEP) ? (uint32_t)mt.lrow : (uint32_t)(a.row_map ? __ldg(a.row_map + mt.slot) : mt.slot);
        };
        PartialSlot* const pbase = a.partials + (long long)mt.slot * a.pstride;
        // lane 1 publishes the result of chunk c (lane 0 is busy issuing copies): self-validating words
        auto publish_chunk = [&](int c, float rm, float rs, int ri, float rk) {
            if (lane == 1) {
                PartialSlot* ps = pbase + c;
                st_relaxed_gpu_u64(&ps->m, tag | (unsigned)__float_as_int(rm));
                st_relaxed_gpu_u64(&ps->s, tag | (unsigned)__float_as_int(rs));
                st_relaxed_gpu_u64(&ps->idx, tag | (unsigned)ri);
                if (SAMPLE) st_relaxed_gpu_u64(&ps->pad, tag | (unsigned)__float_as_int(rk));
            }
        };
        // The unit is complete: `nch` of the row's `total` chunk results are published.  A RELAXED ticket counts
        // them -- no fence anywhere; whoever completes the row merges: the other units' words were stored before
        // their tickets but nothing orders them, so the merger polls until every tag is current (normally the
        // first read).  Lane l folds the chunks l, l + 32, ... in ascending order, then the warp combination:
        // the same order whoever merges and however the row was cut into units.
        auto unit_done = [&](int nch, int total, bool gathered) {
            int* tk = a.tickets + ((MODE == MODE_FLOW) ? (long long)mt.slot * 2 + (tstep & 1) : (long long)mt.slot);
            bool last = true;
            if (nch != total) {
                int t = 0;
                if (lane == 1) t = atomicAdd(tk, nch);
                t = __shfl_sync(FULL, t, 1);
                last = (t + nch == total);
                if (last && lane == 1) atomicExch(tk, 0);  // (an atomic like the adds it is ordered with, not a plain store)
            }
            if (!last) return;
            if (MODE == MODE_FLOW && lane == 0) CD_DBG_MAX(F, dbg_rec, 4);
            [[maybe_unused]] const unsigned ck2 = CD_CLOCK();
            int q0 = 0, q1 = 0;
            if (MODE == MODE_FLOW && lane == 0) {  // how busy the machine is, for the split of the row's next step
                q0 = ld_relaxed_gpu_s32(F->q + FQ_DRAWN) + (int)(gridDim.x * WARPS);  // (+ the static first units)
                q1 = ld_relaxed_gpu_s32(F->q + FQ_PUBLISHED);
            }
            __syncwarp();
            float rm = -INFINITY, rs = 0.0f, rk = -INFINITY;
            int ri = 0x7FFFFFFF;
            constexpr int ROUNDS = MAX_CHUNKS / 32;
            unsigned long long wm[ROUNDS], ws[ROUNDS], wi[ROUNDS], wk[ROUNDS];
            bool ok[ROUNDS];
#pragma unroll
            for (int r = 0; r < ROUNDS; ++r) {  // every load of every round in flight at once
                const int c = r * 32 + lane;
                ok[r] = c >= total;
                wm[r] = ws[r] = wi[r] = wk[r] = 0;
                if (!ok[r]) {
                    wm[r] = ld_relaxed_gpu_u64(&pbase[c].m);
                    ws[r] = ld_relaxed_gpu_u64(&pbase[c].s);
                    wi[r] = ld_relaxed_gpu_u64(&pbase[c].idx);
                    if (SAMPLE) wk[r] = ld_relaxed_gpu_u64(&pbase[c].pad);
                }
            }
            int spins = 0;
            while (true) {
                bool all_ok = true;
#pragma unroll
                for (int r = 0; r < ROUNDS; ++r) {
                    if (!ok[r]) {
                        ok[r] = ((wm[r] >> 32) == gen) && ((ws[r] >> 32) == gen) && ((wi[r] >> 32) == gen) &&
                                (!SAMPLE || (wk[r] >> 32) == gen);
                        if (!ok[r]) {  // a stale word: read the slot again
                            const int c = r * 32 + lane;
                            wm[r] = ld_relaxed_gpu_u64(&pbase[c].m);
                            ws[r] = ld_relaxed_gpu_u64(&pbase[c].s);
                            wi[r] = ld_relaxed_gpu_u64(&pbase[c].idx);
                            if (SAMPLE) wk[r] = ld_relaxed_gpu_u64(&pbase[c].pad);
                            all_ok = false;
                        }
                    }
                }
                if (__all_sync(FULL, all_ok)) break;
                __nanosleep(32);
                if (++spins > MERGE_SPIN_LIMIT) {  // never on a healthy run: fail the call, do not hang
                    if (lane == 0) atomicAdd(MODE == MODE_FLOW ? F->q + FQ_ERRORS : a.ctrs + 2, 1);
                    break;
                }
            }
#pragma unroll
            for (int r = 0; r < ROUNDS; ++r) {
                if (r * 32 + lane < total) {
                    if (SAMPLE) {
                        int dummy = 0;
                        online_combine(rm, rs, dummy, __int_as_float((int)(unsigned)wm[r]), __int_as_float((int)(unsigned)ws[r]), 0);
                        sample_combine(rk, ri, __int_as_float((int)(unsigned)wk[r]), (int)(unsigned)wi[r]);
                    } else {
                        online_combine(rm, rs, ri, __int_as_float((int)(unsigned)wm[r]), __int_as_float((int)(unsigned)ws[r]),
                                       (int)(unsigned)wi[r]);
                    }
                }
            }
            warp_combine_s<SAMPLE>(rm, rs, ri, rk);
            if (MODE == MODE_FLOW && lane == 0) CD_DBG_MAX(F, dbg_rec, 5);
            [[maybe_unused]] const unsigned ck3 = CD_CLOCK();
            if (MODE == MODE_FLOW && lane == 0) CD_DBG_CYC(F, dbg_rec, 11, ck3 - ck2);
            // SAMPLE: the tempered logit of the sampled token is re-read from the logits row
            float ytok = 0.0f;
            if (SAMPLE && rm != -INFINITY) {
                const int tokid = gathered ? __ldg(a.dfa.tok + mt.csr_lo + ri) : ri;
                const unsigned char* rowp = tlogits + (long long)mt.lrow * a.ld_bytes;
                const float xv = (DT == DT_BF16)
                                     ? __uint_as_float(((uint32_t)__ldg(reinterpret_cast<const uint16_t*>(rowp) + tokid)) << 16)
                                     : __ldg(reinterpret_cast<const float*>(rowp) + tokid);
                ytok = __fmul_rn(xv, a.inv_tau);
            }
            finalize_row<MODE>(a, sv, F, mt, rm, rs, ri, lane, gathered, SAMPLE, ytok, __shfl_sync(FULL, q0, 0),
                               __shfl_sync(FULL, q1, 0), units0);
            if (MODE == MODE_FLOW && lane == 0) CD_DBG_CYC(F, dbg_rec, 12, CD_CLOCK() - ck3);
        };

        if (mt.flags & (FLAG_ACCEPT | FLAG_BADSTATE)) {
            // accepted rows never advance; a state outside [0, S) is reported done
            if (fpart == 0) {
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
                        atomicAdd(MODE == MODE_FLOW ? F->q + FQ_ERRORS : a.ctrs + 2, 1);
                        if (MODE != MODE_FLOW && a.hist_tokens) {  // the row leaves the loop here, undone, in the state it has
                            const long long rid = orig_row();
                            a.hist_final_state[rid] = mt.st;
                            a.hist_done[rid] = 0;
                        }
                    }
                }
                // (flow_kernel never holds an accepting row; a row in a state outside [0, S) leaves undone)
                if (MODE == MODE_FLOW) flow_row_leaves(a, sv, *F, mt.lrow, mt.step, mt.st, __uint_as_float(mt.sumbits), 0, lane);
            }
        } else if (GATHER && (mt.flags & FLAG_GATHER)) {
            // unit `fpart` of `fcnt` of a gathered row: the canonical pieces [p0, p1) of the state's CSR row.  Per
            // piece: tokens read coalesced, their logits gathered with GATHER_UNROLL independent loads per lane;
            // idx = position in the CSR row, which ascends with the token id, so "replace on strictly greater"
            // keeps the lowest id
            const int npieces = gather_pieces(mt.csr_len), gp = gather_piece(mt.csr_len);
            const int p0 = (int)(((long long)npieces * fpart) / fcnt), p1 = (int)(((long long)npieces * (fpart + 1)) / fcnt);
            const uint32_t row_key = SAMPLE ? rng_row_key(a.seed_lo, a.seed_hi, orig_row(), (uint32_t)rng_step) : 0u;
            const int* tk = a.dfa.tok + mt.csr_lo;
            const unsigned char* rowp = tlogits + (long long)mt.lrow * a.ld_bytes;
#pragma unroll 1
            for (int p = p0; p < p1; ++p) {
                reset_chains();
                const int j0 = p * gp;
                const int j1 = min(mt.csr_len, j0 + gp);
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
                        if constexpr (SAMPLE)
                            online_update_sample(am[0], as[0], kb, ai[0], fmaxf(x[u], -INFINITY), tc[u], j + 32 * u, a.inv_tau, row_key);
                        else
                            online_update(am[u % NC], as[u % NC], ai[u % NC], fmaxf(x[u], -INFINITY), j + 32 * u);  // NaN -> -inf
                    }
                }
                many_chains = true;
                float rm, rs, rk;
                int ri;
                chunk_result(rm, rs, ri, rk);
                publish_chunk(p, rm, rs, ri, rk);
            }
            __syncwarp();
            if (MODE == MODE_FLOW && lane == 0) CD_DBG_MAX(F, dbg_rec, 3);
            unit_done(p1 - p0, npieces, true);
        } else {
            if (MODE == MODE_FLOW && lane == 0 && (mt.flags & FLAG_FIRST)) CD_DBG_MIN(F, dbg_rec, 7);
            [[maybe_unused]] const unsigned ck0 = CD_CLOCK();
            if (MODE == MODE_FLOW && lane == 0) CD_DBG_CYC(F, dbg_rec, 8, ck0 - (unsigned)mt.pad[1]);
            if (mt.flags & FLAG_FIRST) reset_chains();
            const uint32_t row_key = SAMPLE ? rng_row_key(a.seed_lo, a.seed_hi, orig_row(), (uint32_t)rng_step) : 0u;
            const int t0 = mt.tile * TILE_TOK;
            const uint32_t* mw = reinterpret_cast<const uint32_t*>(ring.mask[cons_stage]);
            const unsigned char* tile = ring.logits[cons_stage];
            // the lane owns the tile's mask words WPL * lane .. WPL * lane + WPL - 1 (consecutive tokens; one
            // vector load from shared memory)
            uint32_t bits[WPL];
            if constexpr (WPL == 4) {
                const uint4 v = reinterpret_cast<const uint4*>(mw)[lane];
                bits[0] = v.x; bits[1] = v.y; bits[2] = v.z; bits[3] = v.w;
            } else if constexpr (WPL == 2) {
                const uint2 v = reinterpret_cast<const uint2*>(mw)[lane];
                bits[0] = v.x; bits[1] = v.y;
            } else {
#pragma unroll
                for (int j = 0; j < WPL; ++j) bits[j] = mw[WPL * lane + j];
            }
            // Sparse tile (at most TILE_LIST_CAP allowed elements -- the normal case of a constrained step): the
            // allowed positions are first compacted across the warp (one exclusive scan of the per-lane popcounts =
            // ascending token order, positions written to a small shared list) and lane l then evaluates exactly the
            // elements of rank l, l + 32, ... (ascending per lane, so "replace on strictly greater" still keeps
            // the lowest id).  Every lane gets its fair share of the tile's allowed elements -- the bit walk below
            // runs as long as the fullest word of any lane -- and only allowed elements cost an evaluation (with
            // sampling: a hash and two logarithms each).
            int cnt = 0;
#pragma unroll
            for (int j = 0; j < WPL; ++j) cnt += __popc(bits[j]);
            int inc = cnt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int up = __shfl_up_sync(FULL, inc, o);
                if (lane >= o) inc += up;
            }
            const int total = __shfl_sync(FULL, inc, 31);
            if (total <= TILE_LIST_CAP) {
                int o = inc - cnt;
#pragma unroll
                for (int j = 0; j < WPL; ++j) {
                    uint32_t b = bits[j];
                    const int e0 = (WPL * lane + j) * 32;
                    while (b != 0u) {
                        ring.list[o++] = (unsigned short)(e0 + __ffs(b) - 1);
                        b &= b - 1u;
                    }
                }
                __syncwarp();
                for (int r = lane; r < total; r += 32) {
                    const int e = ring.list[r];
                    if constexpr (SAMPLE)
                        online_update_sample(am[0], as[0], kb, ai[0], tile_elem<DT>(tile, e), t0 + e, t0 + e, a.inv_tau, row_key);
                    else
                        online_update(am[0], as[0], ai[0], tile_elem<DT>(tile, e), t0 + e);
                }
            } else if constexpr (SAMPLE) {
#pragma unroll
                for (int j = 0; j < WPL; ++j) {
                    // warp-uniform trip count (max popcount over the lanes); idle lanes feed -inf
                    uint32_t b = bits[j];
                    const int e0 = (WPL * lane + j) * 32;
                    while (__any_sync(FULL, b != 0u)) {
                        const bool v = b != 0u;
                        const int e = e0 + (v ? (__ffs(b) - 1) : 0);
                        b &= b - 1u;
                        const float x = v ? tile_elem<DT>(tile, e) : -INFINITY;
                        online_update_sample(am[0], as[0], kb, ai[0], x, t0 + e, t0 + e, a.inv_tau, row_key);
                    }
                }
            } else {
                // dense tile: the lane's WPL words advance together, one chain each: the trip count is the largest
                // popcount of any word of the tile (warp-uniform); chains without a bit left feed -inf
                many_chains = true;
                uint32_t any = 0u;
#pragma unroll
                for (int j = 0; j < WPL; ++j) any |= bits[j];
                while (__any_sync(FULL, any != 0u)) {
                    any = 0u;
#pragma unroll
                    for (int j = 0; j < WPL; ++j) {
                        const uint32_t b = bits[j];
                        const bool v = b != 0u;
                        const int e = (WPL * lane + j) * 32 + (v ? (__ffs(b) - 1) : 0);
                        bits[j] = b & (b - 1u);
                        any |= bits[j];
                        const float x = v ? tile_elem<DT>(tile, e) : -INFINITY;
                        online_update(am[j], as[j], ai[j], x, t0 + e);
                    }
                }
            }
            [[maybe_unused]] const unsigned ck1 = CD_CLOCK();
            if (MODE == MODE_FLOW && lane == 0) CD_DBG_CYC(F, dbg_rec, 9, ck1 - ck0);
            if (mt.flags & FLAG_LAST) {  // the chunk is complete
                float rm, rs, rk;
                int ri;
                chunk_result(rm, rs, ri, rk);
                publish_chunk(fpart, rm, rs, ri, rk);
                if (MODE == MODE_FLOW && lane == 1) CD_DBG_CYC(F, dbg_rec, 10, CD_CLOCK() - ck1);
                if (mt.flags & FLAG_UEND) {
                    if (MODE == MODE_FLOW && lane == 0) CD_DBG_MAX(F, dbg_rec, 3);
                    unit_done(fcnt, Tc, false);
                }
            }
        }
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
            st_release_gpu_s32(L.bar + LB_GO, k1 | (stop << 30));
        }
        int v;
        const unsigned long long t0 = global_timer_ns();
        while (((v = ld_acquire_gpu_s32(L.bar + LB_GO)) & 0x3FFFFFFF) < k1) {
            if (ld_acquire_gpu_s32(L.bar + LB_ABORT) != 0) { v = k1 | (1 << 30); break; }
            if (global_timer_ns() - t0 > LOOP_SPIN_TIMEOUT_NS) {  // never on a healthy device: fail, do not hang
                atomicExch(L.bar + LB_ABORT, 1);
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
// cd_decode_loop without a LIMIT (see FlowArgs).  Every warp is an independent worker that draws units of row
// tasks and returns when every row has left the loop.  There is no block-wide or grid-wide synchronisation
// after the ring set-up, no set-up kernel before the launch and no copy after it.
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
    // Programmatic dependent launch (see step_kernel): this grid may be scheduled while the previous kernel of the
    // stream drains; nothing here reads or writes global memory before that kernel has completed and flushed.
    pdl_launch_dependents();
    pdl_wait();
    const unsigned gen0 = (unsigned)__ldcg(a.ctrs + 3);
    const int par = __ldcg(F.q + FQ_LAUNCHES) & 1;
    StepView sv{};
    sv.gen = gen0;
    sv.trace_t = F.trace_t[par];
    sv.trace_n = F.trace_n[par];
    if (blockIdx.x == 0) {  // this launch's buffers were cleared by the previous one; clear the next one's
        for (int k = threadIdx.x; k <= LOOP_TRACE_STEPS; k += WARPS * 32) {
            F.trace_t[par ^ 1][k] = 0ull;
            F.trace_n[par ^ 1][k] = 0;
        }
        if (threadIdx.x == 0) {
            atomicMax(sv.trace_t + 0, global_timer_ns());
            atomicAdd(sv.trace_n + 0, F.B);
        }
    }
    RingPos rp;
    step_body<DT, WARPS, STAGES, TILE_BYTES, GATHER, SAMPLE, MODE_FLOW>(a, sv, &F, ring, rp, warp, lane);
    // ---------------- last CTA to leave: counters and generation for the next launch, status for the host
    __syncthreads();
    if (threadIdx.x == 0) {
        const int d = atom_add_acq_rel_gpu(a.ctrs + 1, 1);
        if (d == (int)gridDim.x - 1) {
            a.ctrs[1] = 0;
            a.ctrs[3] = (int)(gen0 + (unsigned)a.max_steps + 1u);
            const int steps = __ldcg(sv.trace_n + LOOP_TRACE_STEPS);
            sv.trace_t[steps < LOOP_TRACE_STEPS ? steps : LOOP_TRACE_STEPS] = global_timer_ns();
            const int err = __ldcg(F.q + FQ_ERRORS) + ((__ldcg(F.q + FQ_FINISHED) == F.B) ? 0 : 1);  // every row must have left
            F.q[FQ_DRAWN] = 0;
            F.q[FQ_PUBLISHED] = 0;
            F.q[FQ_FINISHED] = 0;
            F.q[FQ_ERRORS] = 0;
            F.q[FQ_LAUNCHES] = par ^ 1;
            // (sticky until the host reads and clears it: cd_loop_sync reports every loop enqueued since the last one)
            if (err) atomicAdd_system(F.host_status, err);
        }
    }
}

}  // namespace cd
