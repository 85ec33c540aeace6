// cd_aux.cuh -- automaton-store build, transition lookup, compaction and decode-loop
// bookkeeping kernels.
#pragma once
#include "cd_common.cuh"

namespace cd {

// a0: CSR -> packed allowed-token bitmask.  One warp per state; mask is pre-zeroed.
__global__ void build_mask_kernel(const long long* __restrict__ row_ptr, const int* __restrict__ tok,
                                  int S, int Wpad, uint32_t* __restrict__ mask) {
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long s = warp; s < S; s += nwarps) {
        const long long lo = row_ptr[s], hi = row_ptr[s + 1];
        uint32_t* row = mask + s * Wpad;
        for (long long j = lo + lane; j < hi; j += 32) {
            const int t = tok[j];
            atomicOr(row + (t >> 5), 1u << (t & 31));
        }
    }
}

// a4-a5 on their own: one warp per slot, 32-ary search of the sorted CSR row.
__global__ void transition_kernel(DfaDev dfa, const int* __restrict__ token, int* __restrict__ state,
                                  int n, uint8_t* __restrict__ done_out) {
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long i = warp; i < n; i += nwarps) {
        const int st = state[i];
        const int t = token[i];
        int ns = st;
        if (st >= 0 && st < dfa.S) {
            if (t >= 0) {
                const long long j = warp_csr_find(dfa.tok, dfa.row_ptr[st], dfa.row_ptr[st + 1], t, lane);
                if (j >= 0) ns = dfa.next[j];
            }
            if (lane == 0) {
                state[i] = ns;
                done_out[i] = dfa.accepting[ns] ? 1 : 0;
            }
        } else if (lane == 0) {
            done_out[i] = 1;
        }
    }
}

struct CompactArgs {
    const uint8_t* done;
    const int* row_ids_in;  // may be null -> i
    const int* state_in;    // may be null
    int n;
    const int* n_dev;  // if non-null, n is read from the device
    int* row_ids_out;
    int* state_out;
    int* n_active_out;
    // RECORD only (decode loop): per-slot step results -> per-row history
    const int* token;
    const float* logprob;
    int step, max_steps;
    int* tokens_out;
    int* len_out;
    int* final_state_out;
    float* sum_logprob_out;
    uint8_t* done_row_out;
};

// a6: stable stream compaction by one CTA: warp ballot + lane prefix (popc of lower lanes),
// warp totals scanned by warp 0, running base carried across 1024-slot chunks.  n <= 4096 in
// every workload, i.e. at most four chunks.
template <bool RECORD>
__global__ void __launch_bounds__(1024, 1) compact_kernel(const CompactArgs a) {
    __shared__ int warp_off[32];
    __shared__ int chunk_total;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = a.n_dev ? *a.n_dev : a.n;
    int base = 0;
    for (int c0 = 0; c0 < n; c0 += 1024) {
        const int i = c0 + tid;
        const bool valid = i < n;
        const uint8_t d = valid ? a.done[i] : 1;
        const bool keep = valid && (d == 0);
        int rid = 0, st = 0;
        if (valid) {
            rid = a.row_ids_in ? a.row_ids_in[i] : i;
            if (a.state_in) st = a.state_in[i];
        }
        if (RECORD && valid) {
            a.tokens_out[(long long)rid * a.max_steps + a.step] = a.token[i];
            a.len_out[rid] = a.step + 1;
            a.final_state_out[rid] = st;
            a.sum_logprob_out[rid] += a.logprob[i];
            a.done_row_out[rid] = d;
        }
        const unsigned bal = __ballot_sync(FULL, keep);
        const int pre = __popc(bal & ((1u << lane) - 1u));
        if (lane == 0) warp_off[warp] = __popc(bal);
        __syncthreads();
        if (warp == 0) {
            const int v = warp_off[lane];
            int inc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int u = __shfl_up_sync(FULL, inc, o);
                if (lane >= o) inc += u;
            }
            warp_off[lane] = inc - v;  // exclusive
            if (lane == 31) chunk_total = inc;
        }
        __syncthreads();
        if (keep) {
            const int pos = base + warp_off[warp] + pre;
            a.row_ids_out[pos] = rid;
            if (a.state_in) a.state_out[pos] = st;
        }
        base += chunk_total;
        __syncthreads();
    }
    if (tid == 0) *a.n_active_out = base;
}

// a7 set-up: every row starts in the start state with an empty history.
__global__ void loop_init_kernel(int B, int max_steps, int start, int start_accepting, int* row_ids,
                                 int* state, int* n_active, int* tokens_out, int* len_out,
                                 int* final_state_out, float* sum_logprob_out, uint8_t* done_row_out) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long nth = (long long)gridDim.x * blockDim.x;
    for (long long j = tid; j < (long long)B * max_steps; j += nth) tokens_out[j] = -1;
    for (long long r = tid; r < B; r += nth) {
        row_ids[r] = (int)r;
        state[r] = start;
        len_out[r] = 0;
        final_state_out[r] = start;
        sum_logprob_out[r] = 0.0f;
        done_row_out[r] = start_accepting ? 1 : 0;
    }
    if (tid == 0) *n_active = start_accepting ? 0 : B;
}

}  // namespace cd
