/*
 * cd.h -- C ABI of the B200 (sm_100a) batched type-constrained decoding step.
 *
 * What this library computes.  A local-LM query engine applies an LM function
 * with a typed output (boolean, one value of an option set, a regex-shaped
 * value) to every row of a table, one row per prompt (section 2.3.2,
 * L93-L106), and restricts every generation to the strings of that type by
 * masking the logits at each decoding step (section 2.3 "Constrained
 * Decoding", L61; section 7).  Finished sequences leave the running
 * batch (continuous batching, section 4.2).  The paper delegates
 * the step to third-party engines and gives no kernel; the operation is fixed
 * by BASELINE.json north_star:
 *
 *   for each active row i with automaton state s_i and logits row x_i[0..V):
 *     A   = { t : state s_i has a transition on token t }     (allowed set)
 *     m   = max_{t in A} x_i[t]                                (NaN read as -inf)
 *     t*  = min { t in A : x_i[t] == m }                       (ties -> lowest id)
 *     lse = m + log sum_{t in A} exp(x_i[t] - m)               (fp32 accumulate)
 *     logprob = -log sum_{t in A} exp(x_i[t] - m)              (= x_i[t*] - lse)
 *     s_i' = next(s_i, t*)     via the per-state sorted CSR of (token, next)
 *     done_i = accepting[s_i']
 *   then rows with done_i = 1 are removed from the active list, order kept.
 *
 * Conventions
 *   - every entry point returns a cd_status and never throws or aborts; on
 *     error *out arguments are untouched and cd_last_error() (thread local)
 *     describes the failure;
 *   - "DEVICE pointer": memory of the device the automaton was compiled for,
 *     owned by the caller, alive until the stream reaches the call's work;
 *     "HOST pointer": ordinary host memory, read/written before return unless
 *     stated otherwise;
 *   - cd_step, cd_transition and cd_compact are asynchronous on `cuda_stream`
 *     (a cudaStream_t passed as void*; NULL = legacy default stream) and do
 *     not synchronise with the host; cd_decode_loop* synchronise the stream
 *     once before returning;
 *   - the automaton of a handle is immutable after cd_compile_*.  A handle may
 *     be used from several streams and host threads at once: scratch memory is
 *     kept per (handle, stream) and created on the first call that uses that
 *     stream (that first call allocates and therefore synchronises; cd_reserve
 *     does it ahead of time, e.g. before CUDA-graph capture).  The cd_set_*
 *     calls change the handle's SETTINGS (gather thresholds, sampling, LIMIT,
 *     loop mode): every entry point takes a snapshot of the settings when it
 *     starts, under the handle's lock, so a setter may run at any time and
 *     applies to the calls that start after it returns.  Settings are per
 *     handle: two streams that need different settings use two handles (or
 *     order their calls).  cd_set_satisfying overwrites the device copy of the
 *     set in place: do not call it while a loop that uses a LIMIT is running;
 *   - whole-loop kernels (cd_decode_loop, cd_decode_loop_async) occupy every SM and
 *     finish only once each of their thread blocks has run, so two of them never
 *     overlap on one GPU: launched on different streams of one process they run one
 *     after the other (the library orders them; the first time a second stream is
 *     used for a loop on a GPU costs one device synchronisation).  Two PROCESSES
 *     that run loops on the same GPU at the same time are not ordered by anything
 *     and can stall each other until the loop gives up with CD_ERR_INTERNAL: give
 *     each process its own GPU, or use the per-step mode (cd_set_loop_mode);
 *   - logits rows start 16-byte aligned: the base pointer is 16-byte aligned
 *     and ld_elems * sizeof(element) is a multiple of 16; ld_elems >= V.
 *   - there is no CPU fallback: without a CUDA device every call fails with
 *     CD_ERR_CUDA.
 */
#ifndef CD_H_
#define CD_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define CD_API __attribute__((visibility("default")))
#else
#define CD_API
#endif

typedef struct cd_dfa cd_dfa_t; /* opaque; owns device memory */

typedef enum {
    CD_OK = 0,
    CD_ERR_ARG = 1,        /* bad argument: null pointer, negative size, misalignment, ld < V ... */
    CD_ERR_AUTOMATON = 2,  /* malformed CSR                                      */
    CD_ERR_DEAD_STATE = 3, /* a non-accepting state has no transition: argmax over the empty set  */
    CD_ERR_CUDA = 4,       /* a CUDA runtime call failed (message in cd_last_error)               */
    CD_ERR_OOM = 5,        /* host or device allocation failed                                    */
    CD_ERR_INTERNAL = 6    /* a device-side consistency check failed during THIS loop (state out of
                              range, chosen token missing from the CSR) or the persistent loop
                              kernel gave up at a grid barrier; only cd_decode_loop* report it: the
                              affected rows come back with done = 0 in the state they had.  cd_step
                              is asynchronous and reports a slot whose state is outside [0, S)
                              through its outputs only: token -1, logprob 0, done 1, state kept   */
} cd_status;

typedef enum { CD_F32 = 0, CD_BF16 = 1 } cd_dtype;

/*
 * Automaton store (types -> grammar).
 * HOST pointers in, device image out.  The CSR lists, for every state s, the
 * pairs (tok[j], next[j]) for j in [row_ptr[s], row_ptr[s+1]); tok must be
 * strictly increasing inside a state.  The device image holds the CSR, the
 * accepting flags and a packed allowed-token bitmask [S][ceil(V/32) padded to a
 * multiple of 4 words]: bit (t & 31) of word (t >> 5) of row s is set iff state s
 * has a transition on t; pad bits are zero.
 * Errors: CD_ERR_ARG (V < 1, S < 1, null pointer, bad device), CD_ERR_AUTOMATON
 * (row_ptr not non-decreasing from 0, token or next state out of range, tokens
 * not strictly increasing, start out of range), CD_ERR_DEAD_STATE, CD_ERR_OOM,
 * CD_ERR_CUDA.  The input arrays are not referenced after return.
 */
CD_API cd_status cd_compile_dfa(int32_t V, int32_t S, int32_t start, const int64_t* row_ptr /*[S+1]*/,
                         const int32_t* tok /*[nnz]*/, const int32_t* next /*[nnz]*/,
                         const uint8_t* accepting /*[S]*/, int device, cd_dfa_t** out);

/*
 * Sugar for boolean / option-set types (PAPER.md L61 `options`, L110-L133):
 * builds the trie automaton of K labels given as token-id sequences
 * label_tok[label_ptr[k] .. label_ptr[k+1]) (HOST pointers) and compiles it.
 *   eos < 0   a row is finished the first time its state accepts: one
 *             accepting leaf per label, so the final state names the label.  Labels must
 *             be non-empty, distinct and prefix-free (G5: a label extending another would
 *             be unreachable), else CD_ERR_AUTOMATON.
 *   eos >= 0  the EOS / longest-match variant (G4, G5; the paper leaves the
 *             stopping rule to the engine): the language is
 *             { label + [eos] }.  Every state reached by a whole label ("may stop") gets an
 *             eos edge to ONE accepting sink and only the sink accepts, so a label may be a
 *             token-prefix of another ("New York" / "New York City"): in the shorter label's
 *             end state the model either emits eos or goes on.  The decoded row is
 *             label + [eos]; the label is read from the token history.  Labels must be
 *             non-empty, distinct and must not contain eos; eos < V.
 * State numbering (both): 0 = root, trie nodes in insertion order (labels in the given
 * order, token by token), the sink (eos >= 0) last.
 * cd_build_trie is pure host code (no device needed): it writes the number of states and
 * transitions to *S_out / *nnz_out and, where the array pointers are not NULL, the CSR
 * (row_ptr [S+1], tok / next [nnz], accepting [S]; size them from a first call with NULL
 * arrays).  cd_compile_trie builds the same automaton and compiles it (as cd_compile_dfa).
 */
CD_API cd_status cd_build_trie(int32_t V, int32_t K, const int64_t* label_ptr /*[K+1]*/, const int32_t* label_tok,
                        int32_t eos, int32_t* S_out, int64_t* nnz_out, int64_t* row_ptr_out, int32_t* tok_out,
                        int32_t* next_out, uint8_t* accepting_out);
CD_API cd_status cd_compile_trie(int32_t V, int32_t K, const int64_t* label_ptr /*[K+1]*/,
                          const int32_t* label_tok, int32_t eos, int device, cd_dfa_t** out);

/*
 * Sugar for collection types with a quantifier (section 2.3: "If the
 * return_type is a collection, the quantifier argument can be used to apply a regular
 * expression-style modifier to restrict the number of generated items (e.g. {3} for
 * exactly three, {1,5} for between one and five)"): the token-level automaton of
 *     open  item (sep item)^(c-1)  close        for min_items <= c <= max_items
 * (c = 0: open close), every item one of the K labels of cd_compile_trie's form; open, sep,
 * close are token-id sequences (HOST pointers; open may be empty, sep may be empty when
 * max_items == 1, close must not be).  One accepting state, reached by the last token of
 * close.  Deterministic by construction or rejected (CD_ERR_AUTOMATON): labels non-empty,
 * distinct and prefix-free, sep[0] != close[0], and close[0] does not start a label when
 * min_items == 0.  State 0 is the start state.
 * eos >= 0 (the EOS / longest-match variant, see cd_compile_trie): the list is followed by
 * eos -- the accepting state is reached by eos after the last token of close -- and a label
 * may be a token-prefix of another label: an item ends when sep or close follows, so in the
 * shorter label's end state sep[0] / close[0] must not continue a longer label (else
 * CD_ERR_AUTOMATON); eos occurs in no label and in none of open / sep / close.
 * cd_build_list is pure host code (no device needed): it writes the number of states and
 * transitions to *S_out / *nnz_out and, where the array pointers are not NULL, the CSR
 * (row_ptr [S+1], tok / next [nnz], accepting [S]; size them from a first call with NULL
 * arrays).  cd_compile_list builds the same automaton and compiles it (as cd_compile_dfa).
 */
CD_API cd_status cd_build_list(int32_t V, int32_t K, const int64_t* label_ptr, const int32_t* label_tok,
                        const int32_t* open, int32_t n_open, const int32_t* sep, int32_t n_sep,
                        const int32_t* close, int32_t n_close, int32_t min_items, int32_t max_items,
                        int32_t eos, int32_t* S_out, int64_t* nnz_out, int64_t* row_ptr_out, int32_t* tok_out,
                        int32_t* next_out, uint8_t* accepting_out);
CD_API cd_status cd_compile_list(int32_t V, int32_t K, const int64_t* label_ptr, const int32_t* label_tok,
                          const int32_t* open, int32_t n_open, const int32_t* sep, int32_t n_sep,
                          const int32_t* close, int32_t n_close, int32_t min_items, int32_t max_items,
                          int32_t eos, int device, cd_dfa_t** out);

/* Releases the device image and every per-stream scratch area.  NULL is a no-op.
   The caller makes sure no work using the handle is still in flight. */
CD_API void cd_free_dfa(cd_dfa_t* dfa);

/* Shape of a compiled automaton; any out pointer may be NULL. */
CD_API cd_status cd_dfa_info(const cd_dfa_t* dfa, int32_t* V, int32_t* S, int32_t* start, int64_t* nnz,
                      int64_t* mask_bytes);

/*
 * Density-adaptive step.  A masked log-softmax needs only the
 * allowed logits: for a row whose state has at most `max_transitions` transitions
 * cd_step / cd_decode_loop* do not scan the logits row and its bitmask but walk the
 * state's CSR token list and gather exactly the allowed logits.  Outputs are the same
 * as the dense scan's (token, state, done bit-exact; logprob / lse within the same
 * tolerance; the summation order differs).  Rows of both kinds mix in one launch.
 *   max_transitions = 0   dense scan for every state (default: the method
 *                         BASELINE.json north_star states)
 *   max_transitions > 0   gather states with <= max_transitions transitions
 *   max_transitions = -1  automatic threshold from V and the logits dtype
 */
CD_API cd_status cd_set_gather_max(cd_dfa_t* dfa, int32_t max_transitions);

/*
 * Sampling instead of greedy decoding (the paper leaves the decoding rule
 * open -- only a hidden "temperature" of a comparison system is mentioned).
 * With temperature T > 0 cd_step / cd_decode_loop* draw the token of every row from the
 * masked softmax at temperature T by the Gumbel-max rule
 *     y_t = fl32(x_t * fl32(1 / T)),   t* = argmax_{t in A} fl32(y_t + g(row, step, t))
 * (ties -> lowest id), where g is Gumbel(0,1) noise from a counter-based generator keyed
 * by (seed, ORIGINAL row id = row_map[i] or i, step_base + decoding step, token): results
 * do not depend on batch composition, compaction or launch shape, and a rerun with the
 * same seed reproduces them bit for bit.  The generator and the fp32 operation sequence
 * of g are part of the definition (restated in oracle/oracle_cd.c O10).  Outputs:
 * logprob_out = log of the sampled token's probability under the masked softmax of y,
 * lse_out = masked logsumexp of y.  T = 0 (default) restores greedy decoding.  For
 * cd_step the decoding step is step_base; cd_decode_loop* use step_base + k.
 * On the LM-head path (cd_head_*) the same rule applies to the fp32-accumulated logits
 * (bit-identical to the logits path whenever the dot products are exact in fp32).
 */
CD_API cd_status cd_set_sampling(cd_dfa_t* dfa, float temperature, uint64_t seed, int32_t step_base);

/* Creates (or grows) the scratch area of (dfa, cuda_stream) for up to max_rows
   rows, so that later calls on that stream neither allocate nor synchronise. */
CD_API cd_status cd_reserve(const cd_dfa_t* dfa, int32_t max_rows, void* cuda_stream);

/*
 * One constrained step for n active rows: fused allowed-mask
 * read, masked max/argmax, masked logsumexp, CSR transition and accept test, one
 * kernel launch.  All pointers are DEVICE pointers.
 *   logits      [rows, ld_elems] of `dtype`; the row of active slot i is
 *               logits + row_map[i] * ld_elems (row_map == NULL -> row i)
 *   state       [n] in/out: automaton state of slot i, replaced by the next state
 *   token_out   [n] chosen token id; -1 for a slot whose state is already accepting
 *   logprob_out [n] log-probability of the chosen token under the masked softmax
 *   lse_out     [n] masked logsumexp (may be NULL)
 *   done_out    [n] 1 iff the new state is accepting
 * A slot whose state is already accepting does not advance: state unchanged,
 * token -1, logprob 0, lse 0, done 1; a slot whose state is outside [0, S) is
 * reported the same way (nothing else can be said about it without a host
 * synchronisation).  If every allowed logit is -inf (or NaN)
 * the lowest allowed id is chosen and logprob = lse = -inf.  With an allowed
 * +inf logit the lowest such id is chosen; logprob / lse are unspecified.
 * n == 0 is valid and launches nothing.
 */
CD_API cd_status cd_step(const cd_dfa_t* dfa, const void* logits, cd_dtype dtype, int64_t ld_elems,
                  const int32_t* row_map, int32_t* state, int32_t n, int32_t* token_out,
                  float* logprob_out, float* lse_out, uint8_t* done_out, void* cuda_stream);

/*
 * Transition lookup on its own for callers that pick tokens
 * themselves: state[i] <- next(state[i], token[i]); done_out[i] = accepting[new
 * state].  A slot with token[i] < 0 or whose state has no transition on token[i]
 * keeps its state and reports done_out[i] = accepting[state[i]].  DEVICE pointers.
 */
CD_API cd_status cd_transition(const cd_dfa_t* dfa, const int32_t* token, int32_t* state, int32_t n,
                        uint8_t* done_out, void* cuda_stream);

/*
 * Early-exit compaction (finished sequences leave the batch,
 * PAPER.md L412): stable partition keeping the slots with done[i] == 0.
 * Out-of-place.  DEVICE pointers.
 *   row_ids_in  [n] or NULL (NULL -> ids 0..n-1)
 *   state_in    [n] or NULL (then state_out is not written)
 *   row_ids_out [n], state_out [n]: first n_active entries are written
 *   n_active_out device int32
 * Up to 4096 slots one CTA does it (no allocation: the call can be captured in a CUDA
 * graph); longer lists take a single-pass scan over ceil(n / 4096) CTAs with decoupled
 * look-back, whose few bytes of chunk state are stream-ordered scratch (cudaMallocAsync).
 */
CD_API cd_status cd_compact(const uint8_t* done, const int32_t* row_ids_in, const int32_t* state_in,
                     int32_t n, int32_t* row_ids_out, int32_t* state_out, int32_t* n_active_out,
                     void* cuda_stream);

/*
 * cd_compact for callers that must not allocate device memory while they decode.
 *
 * Who that is.  This library usually shares its GPU with the LM server that produces the
 * logits, and such a server claims nearly all of HBM for weights and KV cache when it starts
 * (the paper's set-up runs a quantised model on one 16 GB card).
 * A query engine that decodes next to it has three reasons not to ask the driver for memory
 * per call: the request can fail with out-of-memory although the work needs a few KB; the
 * plain allocator synchronises the whole device, stalling the server's streams; and the
 * stream-ordered allocator that cd_compact uses for long lists needs a memory pool, which some
 * deployments switch off or cap (a pool owned by the engine's own caching allocator, MPS
 * clients with a pinned memory limit, processes running under a fixed cgroup-style HBM
 * budget).  For them the multi-CTA scan of cd_compact exists in a form whose only scratch --
 * one 64-bit word per 4096-slot chunk plus a ticket -- lives in a fixed array inside the
 * library image: CD_COMPACT_NOALLOC_MAX_N / 4096 + 1 words = 32,776 bytes, held by every GPU
 * on which the library is loaded until the process exits.
 *
 * Same arguments, same result as cd_compact (a6: stable partition keeping done[i] == 0; the
 * first *n_active_out entries of row_ids_out / state_out are written; DEVICE pointers, all on
 * one device, the one n_active_out lives on).  This call never calls cudaMalloc, cudaFree,
 * their Async forms or any library routine that allocates: one cudaMemsetAsync over the words
 * it is about to use (they keep the previous call's values and must start at zero) and one
 * kernel launch, both on cuda_stream.
 *
 * Limits and rules that cd_compact does not have:
 *   - n <= CD_COMPACT_NOALLOC_MAX_N (2^24 slots).  A longer list is refused with CD_ERR_ARG and
 *     a message naming the limit; nothing is launched.  Split the list or call cd_compact.
 *   - There is ONE array per GPU and every call on that GPU uses it.  Two calls whose kernels
 *     may run at the same time (different streams, different host threads, two handles --
 *     the array belongs to the library, not to an automaton) race on it and return garbage
 *     or spin: keep calls on one stream, or order them with events.  Calls on different
 *     GPUs do not interact.
 *   - The first call on each GPU resolves the array's device address (cudaGetSymbolAddress,
 *     with that GPU current; this is also when a lazily loaded CUDA module is brought onto the
 *     device).  Make that first call during set-up, outside any stream capture; a call with
 *     n = 0 is enough.
 * Errors: CD_ERR_ARG (as cd_compact, plus n above the limit), CD_ERR_CUDA.
 */
#define CD_COMPACT_NOALLOC_MAX_N (1 << 24)
CD_API cd_status cd_compact_noalloc(const uint8_t* done, const int32_t* row_ids_in, const int32_t* state_in,
                             int32_t n, int32_t* row_ids_out, int32_t* state_out, int32_t* n_active_out,
                             void* cuda_stream);

/*
 * The whole loop: every row starts in the start state; for
 * k = 0 .. max_steps-1 the active rows take one cd_step on step_logits[k]
 * (DEVICE pointers in a HOST array; each [B, ld_elems], indexed by ORIGINAL row
 * id) and finished rows are compacted away.  The active count stays on the
 * device; the stream is synchronised once before returning.  Outputs are DEVICE
 * pointers indexed by original row id:
 *   tokens_out      [B, max_steps] chosen tokens, -1 padded
 *   len_out         [B] tokens generated
 *   final_state_out [B]
 *   sum_logprob_out [B] sum of the chosen tokens' log-probs (fp32)
 *   done_out        [B] 1 iff the row reached an accepting state (0 = truncated)
 * If the start state is accepting every row is done with len 0.
 *
 * How it runs (cd_set_loop_mode):
 *   CD_LOOP_AUTO (default)  ONE kernel launch for the whole loop -- no set-up kernel before it, no
 *       copy after it -- when the device supports it and B <= 32768; the CTAs stay resident and read
 *       step_logits[k] themselves.
 *       - cd_decode_loop: rows are independent, so no row waits for another one.  The
 *         warp that finalises step k of a row publishes the row's step k + 1 (row, next state,
 *         running sum; cut into 1 .. 64 work units) in a device queue, from which every warp draws
 *         work units in order.  While some rows are between two steps
 *         (merge, transition look-up) the others keep the memory system busy: no launch, no counter
 *         reset, no compaction pass and no barrier between steps.  The active set never exists as a
 *         list; the outputs are indexed by original row id, so the results are those of the stable
 *         compaction of a6.
 *       - cd_decode_loop_limit (and cd_set_limit): a LIMIT is defined step by step over ALL rows, so
 *         the steps run in lock-step: one cooperative launch, a grid barrier after every step, the
 *         active set a bitmap over original row ids (slot i of a step = its i-th set bit).
 *       Otherwise, and for the host-buffer and callback forms (whose step inputs appear between
 *       steps), the loop is one cd_step-like launch per decoding step with the compaction fused
 *       into the step kernel's last CTA.
 *   CD_LOOP_BARRIER         the lock-step persistent kernel also without a LIMIT.
 *   CD_LOOP_PER_STEP        always one launch per decoding step.
 * All three give the same outputs bit for bit, sum_logprob_out included, and from run to run: the
 * order of a row's fp32 sums is fixed by the row alone (V and the logits type cut it into chunks
 * whose results are folded in a fixed order), never by the batch, the kernel or timing -- in
 * CD_LOOP_AUTO a row step is cut into more work units when warps are waiting for work and into
 * fewer when the machine is busy, which does not change the result.  For the same reason
 * logprob_out / lse_out of cd_step do not depend on n, row_map or the other slots of the call.
 * (Per-step timings of the last persistent loop: cd_loop_trace in cd_diag.h.)
 *
 * cd_decode_loop_async is cd_decode_loop without the synchronisation: it only enqueues the loop on
 * cuda_stream and returns (CD_LOOP_AUTO, no LIMIT: exactly one kernel launch).  The outputs are valid
 * once the stream has been synchronised; device-side failures of the loops enqueued on (dfa,
 * cuda_stream) since the last cd_loop_sync are reported by cd_loop_sync, which synchronises the
 * stream.  step_logits (the HOST array) may be reused as soon as the call returns.  Several loops may
 * be enqueued back to back on one stream; loops enqueued on different streams run one after the other
 * (see Conventions: a whole-loop kernel occupies the GPU).
 */
typedef enum { CD_LOOP_AUTO = 0, CD_LOOP_PER_STEP = 1, CD_LOOP_BARRIER = 2 } cd_loop_mode;
CD_API cd_status cd_set_loop_mode(cd_dfa_t* dfa, int32_t mode);
CD_API cd_status cd_decode_loop_async(const cd_dfa_t* dfa, const void* const* step_logits, cd_dtype dtype,
                         int64_t ld_elems, int32_t B, int32_t max_steps, int32_t* tokens_out,
                         int32_t* len_out, int32_t* final_state_out, float* sum_logprob_out,
                         uint8_t* done_out, void* cuda_stream);
CD_API cd_status cd_loop_sync(const cd_dfa_t* dfa, void* cuda_stream);
CD_API cd_status cd_decode_loop(const cd_dfa_t* dfa, const void* const* step_logits, cd_dtype dtype,
                         int64_t ld_elems, int32_t B, int32_t max_steps, int32_t* tokens_out,
                         int32_t* len_out, int32_t* final_state_out, float* sum_logprob_out,
                         uint8_t* done_out, void* cuda_stream);

/*
 * LIMIT early exit (section 2.4 "Early Exiting",
 * L152-L154: with a LIMIT the LM function "may terminate as soon as the required
 * number of rows is satisfied ... a cancel event is issued and all outstanding
 * generation requests are terminated").
 * cd_set_satisfying marks the accepting states whose value satisfies the query's
 * predicate (HOST u8[S], copied; e.g. the leaf of the label TRUE for `... = TRUE`;
 * NULL clears).
 * cd_decode_loop_limit is cd_decode_loop with a device counter *satisfied_inout
 * (DEVICE int32, shared by the calls of one query, one call per batch of the
 * table; the caller zeroes it first): every row that reaches an accepting state s
 * with satisfying[s] != 0 adds 1.  If the counter is >= limit at entry no row
 * takes a step (len 0, done 0).  After each decoding step, once the counter has
 * reached limit, every row still active is cancelled: it keeps the tokens it has,
 * done_out = 0, final_state_out = the state it stopped in.  Rows that finish in
 * the same step are all kept, so the counter may end above limit (the caller
 * keeps the first `limit` in row order).  The remaining step launches find an
 * empty active list and do no work.
 * Errors: as cd_decode_loop; CD_ERR_ARG if cd_set_satisfying was not called,
 * satisfied_inout is NULL or limit < 0.
 */
CD_API cd_status cd_set_satisfying(cd_dfa_t* dfa, const uint8_t* satisfying /*[S] or NULL*/);
CD_API cd_status cd_decode_loop_limit(const cd_dfa_t* dfa, const void* const* step_logits, cd_dtype dtype,
                               int64_t ld_elems, int32_t B, int32_t max_steps, int32_t* tokens_out,
                               int32_t* len_out, int32_t* final_state_out, float* sum_logprob_out,
                               uint8_t* done_out, int32_t limit, int32_t* satisfied_inout,
                               void* cuda_stream);

/*
 * LIMIT early exit for every loop entry point: after cd_set_limit(dfa, limit, satisfied)
 * (satisfied: DEVICE int32 owned by the caller, shared by the calls of one query; needs
 * cd_set_satisfying) cd_decode_loop, cd_decode_loop_host, cd_decode_loop_cb and the
 * cd_head_decode_loop* family all behave as cd_decode_loop_limit does.  satisfied == NULL
 * clears it.
 */
CD_API cd_status cd_set_limit(cd_dfa_t* dfa, int32_t limit, int32_t* satisfied_inout);

/*
 * Same loop with HOST buffers end to end: step_logits_host[k] are HOST arrays
 * (pinned memory gives full PCIe rate), the five outputs are HOST arrays.  Early
 * exit reaches the PCIe link: before step k the host reads the compacted active
 * list and copies only the rows still active (runs of consecutive rows as one
 * copy) into a compact device staging buffer kept in the (handle, stream) scratch
 * area, so a loop moves (row-steps * ld_elems * sizeof) bytes instead of
 * (steps * B * ld_elems * sizeof); copying stops as soon as no row is active.
 * With pinned, device-mapped buffers (cudaHostAlloc / cudaHostRegister under unified
 * addressing) nothing is read back between steps: a kernel pulls the active rows over the
 * link.  With the density-adaptive step switched on (cd_set_gather_max != 0) and such buffers,
 * when EVERY state of the automaton may be gathered -- at most max_transitions transitions, or,
 * for -1 (automatic), at most V / 32 -- nothing is staged at all: the step kernel reads the
 * allowed logits of the active rows straight from the host buffers, one 32-byte sector each
 * (configs[4]: 42 KB per row-step instead of 512 KB).  Same outputs either way.
 */
CD_API cd_status cd_decode_loop_host(const cd_dfa_t* dfa, const void* const* step_logits_host,
                              cd_dtype dtype, int64_t ld_elems, int32_t B, int32_t max_steps,
                              int32_t* tokens_out, int32_t* len_out, int32_t* final_state_out,
                              float* sum_logprob_out, uint8_t* done_out, void* cuda_stream);

/*
 * The constrained step fused with the LM head.  The whole cost of the
 * step is the logits tensor, and the paper's point is that constrained decoding should
 * cost nothing next to the model forward (section 5), so the step is
 * defined directly on what produces the logits:
 *     x_i[t] = sum_{h < H} hidden_i[h] * W[t][h]          (LM head, no bias)
 * followed by exactly the step of cd_step on x_i.  The logit is the dot product of the
 * stored bf16 values accumulated in fp32 (tensor-core accumulation order); it is never
 * rounded to a storage type and never written to HBM.  All pointers are DEVICE pointers.
 *   hidden      [rows, ldh_elems] bf16, final hidden states; the row of active slot i is
 *               hidden + row_map[i] * ldh_elems (row_map == NULL -> row i)
 *   W           [V, ldw_elems] bf16, row t = output embedding of token t
 *   H           hidden size, a positive multiple of 8; ldh_elems, ldw_elems >= H and
 *               multiples of 8; both base pointers 16-byte aligned
 *   state, n, token_out, logprob_out, lse_out (may be NULL), done_out: as cd_step
 * Rows whose state has few transitions (boolean / option-set types) form only their
 * allowed logits as gathered dot products; the others go through a dense tcgen05
 * contraction whose epilogue applies each row's allowed-token bitmask
 * (cd_set_head_gather_max: 0 = dense for every state, > 0 = gather states with at most
 * that many transitions, -1 = automatic, the default: states with fewer than V / 300
 * transitions are gathered, and when the remaining rows of a call together touch fewer than
 * 0.8 V rows of W -- a late step of an early-exit loop -- they are gathered too instead of
 * streaming all of W for a handful of rows).  A gathered row is cut into pieces of >= 128
 * transitions, one CTA each, so a few rows of thousands of transitions still spread over
 * the whole machine.  Results agree with cd_step on
 * exactly computed logits: token, state and done are identical whenever the best
 * allowed logit leads the runner-up by more than the fp32 accumulation error (always,
 * when the dot products are exact in fp32); logprob / lse within that error.
 * Errors: CD_ERR_ARG (NULL pointer, bad H / stride / alignment), CD_ERR_CUDA, CD_ERR_OOM.
 */
CD_API cd_status cd_set_head_gather_max(cd_dfa_t* dfa, int32_t max_transitions);
CD_API cd_status cd_head_step(const cd_dfa_t* dfa, const void* hidden, int64_t ldh_elems, const void* W,
                       int64_t ldw_elems, int32_t H, const int32_t* row_map, int32_t* state, int32_t n,
                       int32_t* token_out, float* logprob_out, float* lse_out, uint8_t* done_out,
                       void* cuda_stream);

/*
 * The decode loop on top of cd_head_step (cd_decode_loop with the LM head fused in):
 * step_hidden[k] (DEVICE pointers in a HOST array) are the final hidden states of
 * decoding step k, [B, ldh_elems] bf16 indexed by ORIGINAL row id -- the output of the
 * model forward, which is outside this library.  Outputs and semantics as
 * cd_decode_loop; the active count stays on the device; the stream is synchronised once
 * before returning.
 */
CD_API cd_status cd_head_decode_loop(const cd_dfa_t* dfa, const void* const* step_hidden, int64_t ldh_elems,
                              const void* W, int64_t ldw_elems, int32_t H, int32_t B, int32_t max_steps,
                              int32_t* tokens_out, int32_t* len_out, int32_t* final_state_out,
                              float* sum_logprob_out, uint8_t* done_out, void* cuda_stream);

/*
 * Early deduplication (section 2.4 "Early Deduplication of
 * Database Values", L156): "the input set is deduplicated via a SELECT DISTINCT clause,
 * and the mapped outputs are then aligned to the original table via a LEFT JOIN", which
 * cuts the number of generations by the duplication factor N / |dom|.
 * cd_dedup: keys [N] (DEVICE int64: interned value ids or hashes of the, possibly
 * multi-column, input values; every int64 value is a valid key).  Distinct values are
 * listed in order of first occurrence:
 *   distinct_rows_out [N]  DEVICE; entry p = row id of the first row carrying the p-th
 *                          distinct value (ascending); the first *n_distinct_out are written
 *   rep_out           [N]  DEVICE; rep[i] = p with keys[distinct_rows[p]] == keys[i]
 *   n_distinct_out         DEVICE int32
 * The caller decodes the rows distinct_rows[0 .. n_distinct) only (cd_decode_loop /
 * cd_head_decode_loop on logits or hidden states of those rows) and broadcasts the results
 * back with cd_join_results: out[i] = in[rep[i]] for the five loop outputs (tokens
 * [., max_steps]); an output pointer may be NULL to skip it.  Asynchronous on cuda_stream;
 * scratch is stream-ordered (cudaMallocAsync).  N <= 2^30 per call.  Errors: CD_ERR_ARG, CD_ERR_CUDA,
 * CD_ERR_OOM.
 */
CD_API cd_status cd_dedup(const int64_t* keys, int32_t N, int32_t* rep_out, int32_t* distinct_rows_out,
                   int32_t* n_distinct_out, void* cuda_stream);
CD_API cd_status cd_join_results(const int32_t* rep, int32_t N, int32_t max_steps, const int32_t* tokens_d,
                          const int32_t* len_d, const int32_t* final_state_d, const float* sum_logprob_d,
                          const uint8_t* done_d, int32_t* tokens_out, int32_t* len_out,
                          int32_t* final_state_out, float* sum_logprob_out, uint8_t* done_out,
                          void* cuda_stream);

/*
 * Cascade filtering (section 2.4): with conjunctive LM
 * predicates "subsequent functions only process rows of data which satisfied all preceding
 * predicates".  Given the decode results of one predicate (final_state, done: DEVICE [N])
 * and the satisfying set of cd_set_satisfying, writes the ids of the rows that finished in
 * a satisfying state, order kept (row_ids_in [N] or NULL -> 0..N-1), to row_ids_out [N] and
 * their number to *n_out (DEVICE int32): the active list of the next predicate's loop.
 */
CD_API cd_status cd_filter_rows(const cd_dfa_t* dfa, const int32_t* final_state, const uint8_t* done,
                         const int32_t* row_ids_in, int32_t N, int32_t* row_ids_out, int32_t* n_out,
                         void* cuda_stream);

/*
 * cd_head_decode_loop with HOST buffers end to end: step_hidden_host[k] are HOST arrays
 * [B, ldh_elems] bf16 (pinned memory lets the copies overlap the kernels), W stays a DEVICE
 * pointer (the weights live on the GPU), the five outputs are HOST arrays.  What crosses
 * PCIe per step is B * ldh_elems * 2 bytes of hidden states instead of B * V logits.
 */
CD_API cd_status cd_head_decode_loop_host(const cd_dfa_t* dfa, const void* const* step_hidden_host,
                                   int64_t ldh_elems, const void* W, int64_t ldw_elems, int32_t H, int32_t B,
                                   int32_t max_steps, int32_t* tokens_out, int32_t* len_out,
                                   int32_t* final_state_out, float* sum_logprob_out, uint8_t* done_out,
                                   void* cuda_stream);

/*
 * Callback forms of the loops ("how a real LM forward would plug in").  Before
 * decoding step k the library calls, on the calling host thread,
 *     next_logits(user, k, d_row_ids, d_n_active, n_upper, &logits, &ld_elems, &by_slot)
 * with DEVICE pointers to the current active list (original row ids of the active slots,
 * ascending; *d_n_active of them, at most n_upper = B) -- valid for work enqueued on
 * cuda_stream.  The callback enqueues whatever produces step k's logits (the model forward
 * over the active rows) on the same stream, without synchronising, and returns the DEVICE
 * buffer: *by_slot != 0 means row i of the buffer belongs to active slot i (a compact batch,
 * what a forward over the active rows yields), 0 means rows are indexed by original row id.
 * A non-zero return value aborts the loop with CD_ERR_ARG.  The buffer must stay valid
 * until the loop returns.  Everything else as cd_decode_loop / cd_head_decode_loop (for the
 * head form the callback returns hidden states [., ldh_elems] bf16).
 */
typedef int (*cd_next_logits_fn)(void* user, int32_t step, const int32_t* d_row_ids, const int32_t* d_n_active,
                                 int32_t n_upper, const void** logits_out, int64_t* ld_elems_out,
                                 int32_t* by_slot_out);
typedef cd_next_logits_fn cd_next_hidden_fn;
CD_API cd_status cd_decode_loop_cb(const cd_dfa_t* dfa, cd_next_logits_fn next_logits, void* user, cd_dtype dtype,
                            int32_t B, int32_t max_steps, int32_t* tokens_out, int32_t* len_out,
                            int32_t* final_state_out, float* sum_logprob_out, uint8_t* done_out,
                            void* cuda_stream);
CD_API cd_status cd_head_decode_loop_cb(const cd_dfa_t* dfa, cd_next_hidden_fn next_hidden, void* user, const void* W,
                                 int64_t ldw_elems, int32_t H, int32_t B, int32_t max_steps,
                                 int32_t* tokens_out, int32_t* len_out, int32_t* final_state_out,
                                 float* sum_logprob_out, uint8_t* done_out, void* cuda_stream);

/* Message of the last failure on the calling thread ("" if none). */
CD_API const char* cd_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CD_H_ */
