/*
 * oracle_cd.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU definition of the batched type-constrained
 * decoding step (BASELINE.json north_star).  It
 * exists so that the CUDA path can be checked against something that a reader
 * can compare with the text by eye.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or helper with paper_2606_31808_b200/ and
 * neither side includes the other.
 *
 * What the paper fixes:
 *   - every LM-function generation is restricted to the strings of its
 *     return_type / options set ("constrained decoding ... guaranteeing
 *     adherence to datatype structures", section 2.3);
 *   - the restriction is applied as a mask at the decoding level (section 7,
 *     L458);
 *   - one database row in, one value out (section 2.3.2);
 *   - finished sequences leave the batch (continuous batching, section 4.2,
 *     L412-L414).
 * The paper gives no kernel, layout or equation for the step; the precise
 * definition below is BASELINE.json north_star's: masked max /
 * argmax with ties to the lowest token id, masked logsumexp, CSR transition,
 * accept test, stable early-exit compaction.
 *
 * Representation choices made ON PURPOSE differently from the GPU path: the
 * oracle never builds a bitmask; membership is "token appears in the state's
 * CSR row"; transition lookup is a linear scan; sums are double precision in
 * ascending token order.
 *
 * Pins: tests/test_oracle_pins.py (library log_softmax/argmax on the all-ones
 * automaton, closed forms, brute force on tiny vocabularies, trie language
 * enumeration, hand-computed config c0, invariants).
 * Parity unpinned: log-prob / lse values when an allowed logit is +inf
 * -- only "token is the lowest-id +inf" is defined.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { ORC_OK = 0, ORC_ERR_ARG = 1, ORC_ERR_AUTOMATON = 2, ORC_ERR_DEAD_STATE = 3 };
enum { ORC_F32 = 0, ORC_BF16 = 1 };

/* O1: what a valid automaton is. */
int orc_validate(int32_t V, int32_t S, int32_t start, const int64_t *row_ptr, const int32_t *tok,
                 const int32_t *next, const uint8_t *accepting)
{
    if (V <= 0 || S <= 0 || !row_ptr || !accepting) return ORC_ERR_ARG;
    if (start < 0 || start >= S) return ORC_ERR_AUTOMATON;
    if (row_ptr[0] != 0) return ORC_ERR_AUTOMATON;
    for (int32_t s = 0; s < S; ++s)
        if (row_ptr[s + 1] < row_ptr[s]) return ORC_ERR_AUTOMATON;
    if (row_ptr[S] > 0 && (!tok || !next)) return ORC_ERR_ARG;
    for (int32_t s = 0; s < S; ++s) {
        for (int64_t j = row_ptr[s]; j < row_ptr[s + 1]; ++j) {
            if (tok[j] < 0 || tok[j] >= V) return ORC_ERR_AUTOMATON;
            if (next[j] < 0 || next[j] >= S) return ORC_ERR_AUTOMATON;
            if (j > row_ptr[s] && tok[j] <= tok[j - 1]) return ORC_ERR_AUTOMATON;
        }
    }
    /* argmax over the empty set is undefined: a state with no way out must accept */
    for (int32_t s = 0; s < S; ++s)
        if (row_ptr[s + 1] == row_ptr[s] && !accepting[s]) return ORC_ERR_DEAD_STATE;
    return ORC_OK;
}

/* O2.2: widen a stored logit to fp32 exactly; NaN is read as -inf (G6). */
static float widen(const void *row, int dtype, int64_t t)
{
    float x;
    if (dtype == ORC_BF16) {
        uint32_t bits = ((uint32_t)((const uint16_t *)row)[t]) << 16;
        memcpy(&x, &bits, 4);
    } else {
        x = ((const float *)row)[t];
    }
    if (x != x) x = -INFINITY;
    return x;
}

/*
 * O2: one constrained step for n active rows.  The logits row of slot i is
 * logits + row_map[i]*ld (row_map == NULL -> i).  state[] is updated in place.
 */
int orc_step(int32_t V, int32_t S, const int64_t *row_ptr, const int32_t *tok, const int32_t *next,
             const uint8_t *accepting, const void *logits, int dtype, int64_t ld,
             const int32_t *row_map, int32_t *state, int32_t n, int32_t *token_out,
             double *logprob_out, double *lse_out, uint8_t *done_out)
{
    if (n < 0 || ld < V || (dtype != ORC_F32 && dtype != ORC_BF16)) return ORC_ERR_ARG;
    const int64_t esz = dtype == ORC_BF16 ? 2 : 4;
    for (int32_t i = 0; i < n; ++i) {
        const int32_t s = state[i];
        if (s < 0 || s >= S) return ORC_ERR_ARG;
        /* O2.1: accepted rows never advance */
        if (accepting[s]) {
            token_out[i] = -1;
            logprob_out[i] = 0.0;
            lse_out[i] = 0.0;
            done_out[i] = 1;
            continue;
        }
        const int64_t r = row_map ? (int64_t)row_map[i] : (int64_t)i;
        const char *row = (const char *)logits + r * ld * esz;
        const int64_t lo = row_ptr[s], hi = row_ptr[s + 1];

        /* O2.3: m = max over allowed, t* = lowest id attaining it (ascending
           scan, replace on strictly greater only).  If every allowed logit is
           -inf the lowest allowed id is kept (G6). */
        float m = -INFINITY;
        int32_t tstar = tok[lo];
        for (int64_t j = lo; j < hi; ++j) {
            const float x = widen(row, dtype, tok[j]);
            if (x > m) {
                m = x;
                tstar = tok[j];
            }
        }

        /* O2.4: sum over allowed of exp(x - m), double, ascending id */
        double sum = 0.0;
        for (int64_t j = lo; j < hi; ++j) {
            const float x = widen(row, dtype, tok[j]);
            if (x == -INFINITY) continue; /* contributes exactly 0 */
            sum += exp((double)x - (double)m);
        }
        if (m == -INFINITY) {
            lse_out[i] = -INFINITY;
            logprob_out[i] = -INFINITY;
        } else {
            lse_out[i] = (double)m + log(sum);
            logprob_out[i] = -log(sum); /* log p(t*) = x_t* - lse = -log(sum); never m - lse */
        }

        /* O2.5: transition by linear scan, then the accept test */
        int32_t ns = -1;
        for (int64_t j = lo; j < hi; ++j)
            if (tok[j] == tstar) {
                ns = next[j];
                break;
            }
        token_out[i] = tstar;
        state[i] = ns;
        done_out[i] = accepting[ns] ? 1 : 0;
    }
    return ORC_OK;
}

/* O3: stable removal of finished rows.  row_ids_in == NULL means 0..n-1. */
int orc_compact(const uint8_t *done, const int32_t *row_ids_in, const int32_t *state_in, int32_t n,
                int32_t *row_ids_out, int32_t *state_out, int32_t *n_active_out)
{
    if (n < 0) return ORC_ERR_ARG;
    int32_t k = 0;
    for (int32_t i = 0; i < n; ++i) {
        if (done[i]) continue;
        row_ids_out[k] = row_ids_in ? row_ids_in[i] : i;
        if (state_in && state_out) state_out[k] = state_in[i];
        ++k;
    }
    *n_active_out = k;
    return ORC_OK;
}

/*
 * O4: the whole loop.  step_logits[k] is a [B, ld] array indexed by ORIGINAL
 * row id.  tokens_out is [B, max_steps], -1 padded.  n_active_hist (optional,
 * [max_steps]) receives the number of rows each step processed.
 */
/*
 * O5 (section 2.4 "Early Exiting", L152-L154): with a LIMIT the
 * LM function "may terminate as soon as the required number of rows is satisfied" and
 * outstanding generations are cancelled, "no unnecessary tokens are generated".  Reading
 * (N3): a row satisfies when it reaches an accepting state s with
 * satisfying[s] != 0 (e.g. the leaf of the label TRUE for `... = TRUE`).  *satisfied counts
 * such rows across calls (one call per batch of the table).  If *satisfied >= limit at
 * entry no row takes a step.  After every step the rows that finished in it are counted
 * (all of them: rows finishing in the same step are all kept); once *satisfied >= limit
 * every row still active is cancelled: it keeps the tokens it has, done = 0.
 * satisfying == NULL means no limit (plain O4).
 */
int orc_decode_loop_limit(int32_t V, int32_t S, int32_t start, const int64_t *row_ptr, const int32_t *tok,
                          const int32_t *next, const uint8_t *accepting, const void *const *step_logits,
                          int dtype, int64_t ld, int32_t B, int32_t max_steps, int32_t *tokens_out,
                          int32_t *len_out, int32_t *final_state_out, double *sum_logprob_out,
                          uint8_t *done_out, int32_t *n_active_hist, const uint8_t *satisfying,
                          int32_t limit, int32_t *satisfied)
{
    if (B < 0 || max_steps < 0) return ORC_ERR_ARG;
    if (satisfying && !satisfied) return ORC_ERR_ARG;
    int32_t *ids = (int32_t *)malloc(sizeof(int32_t) * (size_t)(B + 1) * 6);
    double *lp = (double *)malloc(sizeof(double) * (size_t)(B + 1) * 2);
    uint8_t *dn = (uint8_t *)malloc((size_t)B + 1);
    if (!ids || !lp || !dn) {
        free(ids); free(lp); free(dn);
        return ORC_ERR_ARG;
    }
    int32_t *st = ids + (B + 1), *ids2 = ids + 2 * (B + 1), *st2 = ids + 3 * (B + 1),
            *tk = ids + 4 * (B + 1);
    double *lse = lp + (B + 1);
    for (int32_t r = 0; r < B; ++r) {
        for (int32_t k = 0; k < max_steps; ++k) tokens_out[(int64_t)r * max_steps + k] = -1;
        len_out[r] = 0;
        final_state_out[r] = start;
        sum_logprob_out[r] = 0.0;
        done_out[r] = accepting[start] ? 1 : 0; /* G13 */
    }
    if (n_active_hist)
        for (int32_t k = 0; k < max_steps; ++k) n_active_hist[k] = 0;
    int32_t n = 0;
    const int exhausted_at_entry = satisfying && *satisfied >= limit;
    if (!accepting[start] && !exhausted_at_entry)
        for (int32_t r = 0; r < B; ++r) {
            ids[n] = r;
            st[n] = start;
            ++n;
        }
    int rc = ORC_OK;
    for (int32_t k = 0; k < max_steps && n > 0; ++k) {
        if (n_active_hist) n_active_hist[k] = n;
        rc = orc_step(V, S, row_ptr, tok, next, accepting, step_logits[k], dtype, ld, ids, st, n, tk,
                      lp, lse, dn);
        if (rc != ORC_OK) break;
        for (int32_t i = 0; i < n; ++i) {
            const int32_t r = ids[i];
            tokens_out[(int64_t)r * max_steps + k] = tk[i];
            len_out[r] = k + 1;
            final_state_out[r] = st[i];
            sum_logprob_out[r] += lp[i];
            done_out[r] = dn[i];
            if (satisfying && dn[i] && satisfying[st[i]]) ++*satisfied;
        }
        if (satisfying && *satisfied >= limit) break; /* cancel every row still active */
        int32_t n2 = 0;
        orc_compact(dn, ids, st, n, ids2, st2, &n2);
        memcpy(ids, ids2, sizeof(int32_t) * (size_t)n2);
        memcpy(st, st2, sizeof(int32_t) * (size_t)n2);
        n = n2;
    }
    free(ids); free(lp); free(dn);
    return rc;
}

/* O4 = O5 without a limit. */
int orc_decode_loop(int32_t V, int32_t S, int32_t start, const int64_t *row_ptr, const int32_t *tok,
                    const int32_t *next, const uint8_t *accepting, const void *const *step_logits,
                    int dtype, int64_t ld, int32_t B, int32_t max_steps, int32_t *tokens_out,
                    int32_t *len_out, int32_t *final_state_out, double *sum_logprob_out,
                    uint8_t *done_out, int32_t *n_active_hist)
{
    return orc_decode_loop_limit(V, S, start, row_ptr, tok, next, accepting, step_logits, dtype, ld, B,
                                 max_steps, tokens_out, len_out, final_state_out, sum_logprob_out,
                                 done_out, n_active_hist, NULL, 0, NULL);
}

/*
 * O6: the constrained step fused with the LM head.  The paper's point
 * is that the constrained step should cost nothing next to the model forward (PAPER.md
 * section 5: "adds little-to-no overhead"); the whole cost of the step is the
 * logits tensor, so the step is defined directly on what produces it:
 *
 *     x_i[t] = sum_{h < H} hidden_i[h] * W[t][h]        (the LM head, no bias)
 *
 * with hidden [rows, ldh] and W [V, ldw] stored as bf16 (row t of W = output embedding
 * of token t), followed by exactly O2 on x_i.  Reading (N2): the logit is the
 * real-number dot product of the stored bf16 values -- it is never rounded to a storage
 * type.  Here: every bf16 widened exactly to double, products and the sum in double,
 * ascending h (H <= 2^20 terms of 16 significant bits each: the double sum is exact to
 * ~1e-13 relative).  Only the allowed tokens' logits are formed (membership = the
 * state's CSR row, as in O2).  NaN products are read as -inf (G6).
 *
 * Outputs as orc_step, plus gap_out[i] = m - (largest allowed logit at another token id),
 * +inf if the state allows one token: a GPU path that accumulates in fp32 may pick a
 * different token only when gap is below its rounding error (tests use it that way).
 */
static double bf16_to_double(uint16_t b)
{
    uint32_t bits = ((uint32_t)b) << 16;
    float x;
    memcpy(&x, &bits, 4);
    return (double)x;
}

/* x = <hidden_row, W[t]> in double, ascending h. */
double orc_head_logit(const uint16_t *hidden_row, const uint16_t *W, int64_t ldw, int32_t H, int32_t t)
{
    const uint16_t *w = W + (int64_t)t * ldw;
    double acc = 0.0;
    for (int32_t h = 0; h < H; ++h) acc += bf16_to_double(hidden_row[h]) * bf16_to_double(w[h]);
    return acc;
}

int orc_head_step(int32_t V, int32_t S, const int64_t *row_ptr, const int32_t *tok, const int32_t *next,
                  const uint8_t *accepting, const uint16_t *hidden, int64_t ldh, const uint16_t *W,
                  int64_t ldw, int32_t H, const int32_t *row_map, int32_t *state, int32_t n,
                  int32_t *token_out, double *logprob_out, double *lse_out, uint8_t *done_out,
                  double *gap_out)
{
    if (n < 0 || H < 1 || ldh < H || ldw < H || V < 1) return ORC_ERR_ARG;
    for (int32_t i = 0; i < n; ++i) {
        const int32_t s = state[i];
        if (s < 0 || s >= S) return ORC_ERR_ARG;
        if (accepting[s]) { /* O2.1 */
            token_out[i] = -1;
            logprob_out[i] = 0.0;
            lse_out[i] = 0.0;
            done_out[i] = 1;
            if (gap_out) gap_out[i] = INFINITY;
            continue;
        }
        const int64_t r = row_map ? (int64_t)row_map[i] : (int64_t)i;
        const uint16_t *hrow = hidden + r * ldh;
        const int64_t lo = row_ptr[s], hi = row_ptr[s + 1];
        double *x = (double *)malloc(sizeof(double) * (size_t)(hi - lo));
        if (!x) return ORC_ERR_ARG;
        for (int64_t j = lo; j < hi; ++j) {
            double v = orc_head_logit(hrow, W, ldw, H, tok[j]);
            if (v != v) v = -INFINITY;
            x[j - lo] = v;
        }
        /* O2.3 on x: ascending id, replace on strictly greater */
        double m = -INFINITY;
        int64_t jstar = lo;
        for (int64_t j = lo; j < hi; ++j)
            if (x[j - lo] > m) {
                m = x[j - lo];
                jstar = j;
            }
        double second = -INFINITY;
        for (int64_t j = lo; j < hi; ++j)
            if (j != jstar && x[j - lo] > second) second = x[j - lo];
        /* O2.4 */
        double sum = 0.0;
        for (int64_t j = lo; j < hi; ++j) {
            if (x[j - lo] == -INFINITY) continue;
            sum += exp(x[j - lo] - m);
        }
        if (m == -INFINITY) {
            lse_out[i] = -INFINITY;
            logprob_out[i] = -INFINITY;
        } else {
            lse_out[i] = m + log(sum);
            logprob_out[i] = -log(sum);
        }
        if (gap_out) gap_out[i] = (hi - lo > 1) ? m - second : INFINITY;
        free(x);
        /* O2.5 */
        token_out[i] = tok[jstar];
        state[i] = next[jstar];
        done_out[i] = accepting[next[jstar]] ? 1 : 0;
    }
    return ORC_OK;
}

/*
 * O7: the decode loop (O4) on top of the LM-head step (O6): step_hidden[k] is the [B, ldh]
 * bf16 array of final hidden states of decoding step k, indexed by ORIGINAL row id (the
 * model forward that produces it is outside the path).  Everything else as O4.
 */
int orc_head_decode_loop(int32_t V, int32_t S, int32_t start, const int64_t *row_ptr, const int32_t *tok,
                         const int32_t *next, const uint8_t *accepting, const uint16_t *const *step_hidden,
                         int64_t ldh, const uint16_t *W, int64_t ldw, int32_t H, int32_t B, int32_t max_steps,
                         int32_t *tokens_out, int32_t *len_out, int32_t *final_state_out,
                         double *sum_logprob_out, uint8_t *done_out, int32_t *n_active_hist)
{
    if (B < 0 || max_steps < 0) return ORC_ERR_ARG;
    int32_t *ids = (int32_t *)malloc(sizeof(int32_t) * (size_t)(B + 1) * 5);
    double *lp = (double *)malloc(sizeof(double) * (size_t)(B + 1) * 2);
    uint8_t *dn = (uint8_t *)malloc((size_t)B + 1);
    if (!ids || !lp || !dn) {
        free(ids); free(lp); free(dn);
        return ORC_ERR_ARG;
    }
    int32_t *st = ids + (B + 1), *ids2 = ids + 2 * (B + 1), *st2 = ids + 3 * (B + 1), *tk = ids + 4 * (B + 1);
    double *lse = lp + (B + 1);
    for (int32_t r = 0; r < B; ++r) {
        for (int32_t k = 0; k < max_steps; ++k) tokens_out[(int64_t)r * max_steps + k] = -1;
        len_out[r] = 0;
        final_state_out[r] = start;
        sum_logprob_out[r] = 0.0;
        done_out[r] = accepting[start] ? 1 : 0;
    }
    int32_t n = 0;
    if (!accepting[start])
        for (int32_t r = 0; r < B; ++r) {
            ids[n] = r;
            st[n] = start;
            ++n;
        }
    int rc = ORC_OK;
    for (int32_t k = 0; k < max_steps; ++k) {
        if (n_active_hist) n_active_hist[k] = n;
        if (n == 0) continue;
        rc = orc_head_step(V, S, row_ptr, tok, next, accepting, step_hidden[k], ldh, W, ldw, H, ids, st, n, tk, lp,
                           lse, dn, NULL);
        if (rc != ORC_OK) break;
        for (int32_t i = 0; i < n; ++i) {
            const int32_t r = ids[i];
            tokens_out[(int64_t)r * max_steps + k] = tk[i];
            len_out[r] = k + 1;
            final_state_out[r] = st[i];
            sum_logprob_out[r] += lp[i];
            done_out[r] = dn[i];
        }
        int32_t n2 = 0;
        orc_compact(dn, ids, st, n, ids2, st2, &n2);
        memcpy(ids, ids2, sizeof(int32_t) * (size_t)n2);
        memcpy(st, st2, sizeof(int32_t) * (size_t)n2);
        n = n2;
    }
    free(ids); free(lp); free(dn);
    return rc;
}

/*
 * O8 (section 2.4 "Early Deduplication of Database Values", L156):
 * "the input set is deduplicated via a SELECT DISTINCT clause, and the mapped outputs are
 * then aligned to the original table via a LEFT JOIN".  Row values are 64-bit keys.
 * Reading (the paper does not order the DISTINCT result): distinct values are listed in
 * order of FIRST OCCURRENCE, which makes the result unique.  distinct_rows[p] = row id of
 * the first row carrying the p-th distinct value; rep[i] = p such that
 * keys[distinct_rows[p]] == keys[i].  Written as the definition: every row scans the list
 * of distinct values found so far.
 */
int orc_dedup(const int64_t *keys, int32_t N, int32_t *rep_out, int32_t *distinct_rows_out, int32_t *n_distinct_out)
{
    if (N < 0) return ORC_ERR_ARG;
    int32_t D = 0;
    for (int32_t i = 0; i < N; ++i) {
        int32_t p = 0;
        while (p < D && keys[distinct_rows_out[p]] != keys[i]) ++p;
        if (p == D) distinct_rows_out[D++] = i;
        rep_out[i] = p;
    }
    *n_distinct_out = D;
    return ORC_OK;
}

/* LEFT JOIN back: row i receives the outputs of distinct value rep[i]. */
int orc_join_results(const int32_t *rep, int32_t N, int32_t max_steps, const int32_t *tokens_d, const int32_t *len_d,
                     const int32_t *fs_d, const double *slp_d, const uint8_t *done_d, int32_t *tokens, int32_t *len,
                     int32_t *fs, double *slp, uint8_t *done)
{
    if (N < 0 || max_steps < 0) return ORC_ERR_ARG;
    for (int32_t i = 0; i < N; ++i) {
        const int32_t r = rep[i];
        for (int32_t k = 0; k < max_steps; ++k) tokens[(int64_t)i * max_steps + k] = tokens_d[(int64_t)r * max_steps + k];
        len[i] = len_d[r];
        fs[i] = fs_d[r];
        slp[i] = slp_d[r];
        done[i] = done_d[r];
    }
    return ORC_OK;
}

/*
 * O9 (section 2.4 "Cascade Filtering", L150): "subsequent functions only process
 * rows of data which satisfied all preceding predicates".  A row satisfies the predicate
 * when it finished (done) in a state of the satisfying set; survivors keep their order.
 * row_ids_in == NULL means 0..N-1.
 */
int orc_filter_rows(const int32_t *final_state, const uint8_t *done, const int32_t *row_ids_in, int32_t N,
                    const uint8_t *satisfying, int32_t S, int32_t *row_ids_out, int32_t *n_out)
{
    if (N < 0) return ORC_ERR_ARG;
    int32_t k = 0;
    for (int32_t i = 0; i < N; ++i) {
        const int32_t s = final_state[i];
        if (done[i] && s >= 0 && s < S && satisfying[s]) row_ids_out[k++] = row_ids_in ? row_ids_in[i] : i;
    }
    *n_out = k;
    return ORC_OK;
}

/*
 * O10: sampling instead of greedy decoding.  The paper leaves the
 * decoding rule open (only a hidden "temperature" of a comparison system is mentioned,
 * PAPER.md L226).  Reading (N5): with temperature T > 0 the token of a row is
 * drawn from the masked softmax of y_t = fl32(x_t * fl32(1/T)) by the Gumbel-max rule
 *     t* = argmax_{t in A} fl32(y_t + g(row, step, t)),   ties -> lowest id,
 * g = -ln(-ln u), u = (2 b + 1) / 2^24, b = top 23 bits of a counter hash of
 * (seed, ORIGINAL row id, step, token).  Because fp32 decides an integer here, the
 * generator and the fp32 operation sequence of g are part of the definition; this file
 * restates them in plain C (every operation a single IEEE-754 fp32 operation: compile
 * with -ffp-contract=off) -- it shares no code with the CUDA path.
 * Outputs: logprob = log softmax(y)[t*] = (y_t* - m) - log(sum), lse = m + log(sum), with
 * sum = sum_{t in A} exp(y_t - m) accumulated in double as in O2.
 */
/* murmur3's 32-bit finalizer (public domain; exported so that a test can hold it against the published vectors) */
uint32_t orc_fmix32(uint32_t h)
{
    h ^= h >> 16;
    h *= 0x85EBCA6Bu;
    h ^= h >> 13;
    h *= 0xC2B2AE35u;
    h ^= h >> 16;
    return h;
}

static uint32_t orc_row_key(uint32_t seed_lo, uint32_t seed_hi, uint32_t row, uint32_t step)
{
    uint32_t h = orc_fmix32(seed_lo ^ (row * 0x9E3779B1u));
    return orc_fmix32(h ^ (step * 0x85EBCA77u) ^ seed_hi);
}

/* ln x for positive normal fp32 from +, *, /, fma: x = m 2^e, m in [sqrt(1/2), sqrt 2),
   ln m = 2 atanh(s), s = (m - 1)/(m + 1), odd series up to s^9. */
float orc_det_logf(float x)
{
    int32_t ix;
    memcpy(&ix, &x, 4);
    const int32_t e = (ix - 0x3F3504F3) >> 23;
    const int32_t im = ix - (int32_t)((uint32_t)e << 23);
    float m;
    memcpy(&m, &im, 4);
    const float f = m + -1.0f;
    const float sden = 2.0f + f;
    const float sq = f / sden;
    const float z = sq * sq;
    float p = fmaf(z, 0.111111111f, 0.142857143f);
    p = fmaf(z, p, 0.2f);
    p = fmaf(z, p, 0.333333333f);
    p = fmaf(z, p, 1.0f);
    const float two_s = 2.0f * sq;
    const float r = two_s * p;
    return fmaf((float)e, 0.693147181f, r);
}

float orc_gumbel(uint32_t seed_lo, uint32_t seed_hi, uint32_t row, uint32_t step, uint32_t tok)
{
    const uint32_t rk = orc_row_key(seed_lo, seed_hi, row, step);
    const uint32_t h = orc_fmix32(orc_fmix32(rk ^ (tok * 0xC2B2AE3Du)) + 0x27D4EB2Fu);
    const float u = (float)(2u * (h >> 9) + 1u) * 5.9604644775390625e-8f;
    const float l1 = -orc_det_logf(u);
    return -orc_det_logf(l1);
}

int orc_sample_step(int32_t V, int32_t S, const int64_t *row_ptr, const int32_t *tok, const int32_t *next,
                    const uint8_t *accepting, const void *logits, int dtype, int64_t ld, const int32_t *row_map,
                    int32_t *state, int32_t n, float temperature, uint64_t seed, int32_t step,
                    int32_t *token_out, double *logprob_out, double *lse_out, uint8_t *done_out)
{
    if (n < 0 || ld < V || (dtype != ORC_F32 && dtype != ORC_BF16) || !(temperature > 0.0f)) return ORC_ERR_ARG;
    const int64_t esz = dtype == ORC_BF16 ? 2 : 4;
    const float inv_tau = 1.0f / temperature;
    const uint32_t seed_lo = (uint32_t)(seed & 0xFFFFFFFFu), seed_hi = (uint32_t)(seed >> 32);
    for (int32_t i = 0; i < n; ++i) {
        const int32_t s = state[i];
        if (s < 0 || s >= S) return ORC_ERR_ARG;
        if (accepting[s]) {
            token_out[i] = -1;
            logprob_out[i] = 0.0;
            lse_out[i] = 0.0;
            done_out[i] = 1;
            continue;
        }
        const int64_t r = row_map ? (int64_t)row_map[i] : (int64_t)i;
        const char *row = (const char *)logits + r * ld * esz;
        const int64_t lo = row_ptr[s], hi = row_ptr[s + 1];
        float m = -INFINITY, kbest = -INFINITY, ybest = -INFINITY;
        int64_t jstar = lo;
        for (int64_t j = lo; j < hi; ++j) {
            const float x = widen(row, dtype, tok[j]); /* NaN -> -inf */
            const float y = x * inv_tau;
            if (y > m) m = y;
            const float g = orc_gumbel(seed_lo, seed_hi, (uint32_t)r, (uint32_t)step, (uint32_t)tok[j]);
            const float key = y + g;
            if (key > kbest) { /* ascending id, strictly greater: ties -> lowest id */
                kbest = key;
                ybest = y;
                jstar = j;
            }
        }
        double sum = 0.0;
        for (int64_t j = lo; j < hi; ++j) {
            const float y = widen(row, dtype, tok[j]) * inv_tau;
            if (y == -INFINITY) continue;
            sum += exp((double)y - (double)m);
        }
        if (m == -INFINITY) { /* every allowed logit -inf: lowest allowed id (G6) */
            jstar = lo;
            lse_out[i] = -INFINITY;
            logprob_out[i] = -INFINITY;
        } else {
            lse_out[i] = (double)m + log(sum);
            logprob_out[i] = ((double)ybest - (double)m) - log(sum);
        }
        token_out[i] = tok[jstar];
        state[i] = next[jstar];
        done_out[i] = accepting[next[jstar]] ? 1 : 0;
    }
    return ORC_OK;
}

/* O4 with O10 as the step: decoding step k uses RNG step step_base + k. */
int orc_sample_decode_loop(int32_t V, int32_t S, int32_t start, const int64_t *row_ptr, const int32_t *tok,
                           const int32_t *next, const uint8_t *accepting, const void *const *step_logits, int dtype,
                           int64_t ld, int32_t B, int32_t max_steps, float temperature, uint64_t seed,
                           int32_t step_base, int32_t *tokens_out, int32_t *len_out, int32_t *final_state_out,
                           double *sum_logprob_out, uint8_t *done_out)
{
    if (B < 0 || max_steps < 0) return ORC_ERR_ARG;
    int32_t *ids = (int32_t *)malloc(sizeof(int32_t) * (size_t)(B + 1) * 5);
    double *lp = (double *)malloc(sizeof(double) * (size_t)(B + 1) * 2);
    uint8_t *dn = (uint8_t *)malloc((size_t)B + 1);
    if (!ids || !lp || !dn) {
        free(ids); free(lp); free(dn);
        return ORC_ERR_ARG;
    }
    int32_t *st = ids + (B + 1), *ids2 = ids + 2 * (B + 1), *st2 = ids + 3 * (B + 1), *tk = ids + 4 * (B + 1);
    double *lse = lp + (B + 1);
    int32_t n = 0;
    for (int32_t r = 0; r < B; ++r) {
        for (int32_t k = 0; k < max_steps; ++k) tokens_out[(int64_t)r * max_steps + k] = -1;
        len_out[r] = 0;
        final_state_out[r] = start;
        sum_logprob_out[r] = 0.0;
        done_out[r] = accepting[start] ? 1 : 0;
        if (!accepting[start]) {
            ids[n] = r;
            st[n] = start;
            ++n;
        }
    }
    int rc = ORC_OK;
    for (int32_t k = 0; k < max_steps && n > 0; ++k) {
        rc = orc_sample_step(V, S, row_ptr, tok, next, accepting, step_logits[k], dtype, ld, ids, st, n, temperature,
                             seed, step_base + k, tk, lp, lse, dn);
        if (rc != ORC_OK) break;
        for (int32_t i = 0; i < n; ++i) {
            const int32_t r = ids[i];
            tokens_out[(int64_t)r * max_steps + k] = tk[i];
            len_out[r] = k + 1;
            final_state_out[r] = st[i];
            sum_logprob_out[r] += lp[i];
            done_out[r] = dn[i];
        }
        int32_t n2 = 0;
        orc_compact(dn, ids, st, n, ids2, st2, &n2);
        memcpy(ids, ids2, sizeof(int32_t) * (size_t)n2);
        memcpy(st, st2, sizeof(int32_t) * (size_t)n2);
        n = n2;
    }
    free(ids); free(lp); free(dn);
    return rc;
}
