// cd_aux.cuh -- automaton-store build, transition lookup, compaction and decode-loop
// bookkeeping kernels.
#pragma once
#include "cd_common.cuh"

namespace cd {

// a0: CSR -> packed allowed-token bitmask, and accepting[next] folded into bit 31 of next[]
// (saves one dependent load per row in the step kernel).  One warp per state; mask pre-zeroed.
__global__ void build_mask_kernel(const long long* __restrict__ row_ptr, const int* __restrict__ tok,
                                  int* __restrict__ next, const uint8_t* __restrict__ accepting,
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
            const int ns = next[j];
            next[j] = ns | (accepting[ns] ? (int)0x80000000 : 0);
        }
    }
}

// a0: per-state prefix counts of the mask bits, one entry per 1024 tokens (32 mask words): the position
// of a token inside its state's CSR row is rank1k[s][t >> 10] + the popcount of the block's words below
// t (cd_step.cuh mask_rank) -- the step kernel finds the transition of its argmax without a search.
// One warp per state.
__global__ void build_rank_kernel(const uint32_t* __restrict__ mask, int S, int Wpad, int nblk, int* __restrict__ rank1k) {
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long s = warp; s < S; s += nwarps) {
        const uint32_t* row = mask + s * Wpad;
        int run = 0;
        for (int b = 0; b < nblk; ++b) {
            const int w = b * 32 + lane;
            int c = (w < Wpad) ? __popc(row[w]) : 0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(FULL, c, o);
            if (lane == 0) rank1k[s * nblk + b] = run;
            run += c;
        }
    }
}

// a4-a5 on their own: one warp per slot, 128-ary search of the sorted CSR row.
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
                if (j >= 0) ns = dfa.next[j] & 0x7FFFFFFF;  // bit 31 carries accepting[next]
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

// a6 as a kernel of its own (cd_compact), n <= one chunk: one CTA of 1024 threads, see block_compact.
__global__ void __launch_bounds__(1024, 1) compact_kernel(const uint8_t* done, const int* row_ids_in,
                                                          const int* state_in, int n, int* row_ids_out,
                                                          int* state_out, int* n_active_out) {
    block_compact(done, row_ids_in, state_in, n, row_ids_out, state_out, n_active_out);
}

// a6 for long lists (cd_compact with n > 4096, cd_dedup's ranking, cd_filter_rows): single-pass stable
// compaction over many CTAs with decoupled look-back.  Chunk c (4096 slots, taken in the order CTAs start:
// a ticket, so a chunk never waits for one that has not started) counts its kept slots, publishes the
// count as {status 1 | aggregate}, walks back over its predecessors' words -- 32 at a time, one per lane --
// until it meets an inclusive prefix {status 2 | prefix}, publishes its own inclusive prefix and writes
// its kept slots at base + local rank.  Value and status share one 64-bit word (single-copy atomic), so
// no fence is needed.  tile_state[0 .. chunks) and *ticket start at zero (cleared by the caller on the
// stream).  rank_out (optional): rank_out[i] = output position of kept slot i (cd_dedup).
constexpr int SCAN_CHUNK = 4096;

__global__ void __launch_bounds__(1024, 1)
compact_lookback_kernel(const uint8_t* __restrict__ done, const int* __restrict__ row_ids_in,
                        const int* __restrict__ state_in, int n, int* __restrict__ row_ids_out,
                        int* __restrict__ state_out, int* __restrict__ n_active_out, int* __restrict__ rank_out,
                        unsigned long long* tile_state, int* ticket) {
    __shared__ int s_warp[32];
    __shared__ int s_chunk, s_base, s_total;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_chunk = atomicAdd(ticket, 1);
    __syncthreads();
    const int chunk = s_chunk;
    const int i0 = chunk * SCAN_CHUNK + 4 * tid;
    int rid[4], st[4];
    bool keep[4];
    const bool vec_ok = ((reinterpret_cast<uintptr_t>(done) & 3) == 0) &&
                        (!row_ids_in || (reinterpret_cast<uintptr_t>(row_ids_in) & 15) == 0) &&
                        (!state_in || (reinterpret_cast<uintptr_t>(state_in) & 15) == 0);
    if (vec_ok && i0 + 3 < n) {
        const uint32_t d4 = *reinterpret_cast<const uint32_t*>(done + i0);
#pragma unroll
        for (int q = 0; q < 4; ++q) keep[q] = ((d4 >> (8 * q)) & 0xFFu) == 0u;
        if (row_ids_in) {
            const int4 r4 = *reinterpret_cast<const int4*>(row_ids_in + i0);
            rid[0] = r4.x; rid[1] = r4.y; rid[2] = r4.z; rid[3] = r4.w;
        } else {
#pragma unroll
            for (int q = 0; q < 4; ++q) rid[q] = i0 + q;
        }
        if (state_in) {
            const int4 s4 = *reinterpret_cast<const int4*>(state_in + i0);
            st[0] = s4.x; st[1] = s4.y; st[2] = s4.z; st[3] = s4.w;
        }
    } else {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int i = i0 + q;
            keep[q] = (i < n) && (done[i] == 0);
            rid[q] = (i < n && row_ids_in) ? row_ids_in[i] : i;
            st[q] = (i < n && state_in) ? state_in[i] : 0;
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
        const int v = s_warp[lane];
        int w = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int u = __shfl_up_sync(FULL, w, o);
            if (lane >= o) w += u;
        }
        s_warp[lane] = w - v;  // exclusive offset of each warp
        const int total = __shfl_sync(FULL, w, 31);
        // decoupled look-back (warp 0)
        int base = 0;
        if (chunk > 0) {
            if (lane == 0) st_relaxed_gpu_u64(tile_state + chunk, (1ull << 32) | (unsigned)total);
            int pred = chunk - 1;
            while (true) {
                const int idx = pred - lane;
                unsigned long long v64 = 2ull << 32;  // before chunk 0: an inclusive prefix of 0
                if (idx >= 0) {
                    do {
                        v64 = ld_relaxed_gpu_u64(tile_state + idx);
                    } while ((v64 >> 32) == 0ull);
                }
                const unsigned incl = __ballot_sync(FULL, (v64 >> 32) == 2ull);
                const int first = incl ? (__ffs(incl) - 1) : 31;  // nearest predecessor holding a prefix
                int part = (lane <= first) ? (int)(unsigned)v64 : 0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(FULL, part, o);
                base += part;
                if (incl) break;
                pred -= 32;
            }
        }
        if (lane == 0) {
            st_relaxed_gpu_u64(tile_state + chunk, (2ull << 32) | (unsigned)(base + total));
            s_base = base;
            s_total = total;
        }
    }
    __syncthreads();
    int pos = s_base + s_warp[warp] + inc - cnt;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        if (keep[q]) {
            row_ids_out[pos] = rid[q];
            if (state_in) state_out[pos] = st[q];
            if (rank_out) rank_out[i0 + q] = pos;
            ++pos;
        }
    }
    if (tid == 0 && (long long)(chunk + 1) * SCAN_CHUNK >= n) *n_active_out = s_base + s_total;
}

// a7 set-up: every row starts in the start state with an empty history.  `ctrs` is the scratch
// area's counter block: the error count is zeroed so that a loop reports its own failures only.
// Per-step loops use (row_ids, state, n_active); the persistent loop (loop_kernel) uses the three
// active-row bitmaps, the two state arrays by row id, the per-step work counters and the barrier words.
struct LoopInitArgs {
    int B, max_steps, start, start_accepting;
    int* row_ids;
    int* state;
    int* n_active;
    int* tokens_out;
    int* len_out;
    int* final_state_out;
    float* sum_logprob_out;
    uint8_t* done_row_out;
    const int* sat_ctr;
    int limit;
    int* ctrs;
    // loop_kernel (all NULL otherwise)
    uint32_t* alive[3];
    int* state2[2];
    int* work;
    int* bar;
};

__global__ void loop_init_kernel(const LoopInitArgs a) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long nth = (long long)gridDim.x * blockDim.x;
    const int B = a.B;
    for (long long j = tid; j < (long long)B * a.max_steps; j += nth) a.tokens_out[j] = -1;
    // LIMIT already satisfied by earlier batches: no row takes a step
    const bool none = a.start_accepting || (a.sat_ctr && *a.sat_ctr >= a.limit);
    for (long long r = tid; r < B; r += nth) {
        if (a.row_ids) a.row_ids[r] = (int)r;
        if (a.state) a.state[r] = a.start;
        if (a.state2[0]) a.state2[0][r] = a.start;
        a.len_out[r] = 0;
        a.final_state_out[r] = a.start;
        a.sum_logprob_out[r] = 0.0f;
        a.done_row_out[r] = a.start_accepting ? 1 : 0;
    }
    if (a.alive[0]) {
        const int nwords = (B + 31) >> 5;
        for (long long w = tid; w < nwords; w += nth) {
            const int rem = B - (int)w * 32;
            a.alive[0][w] = none ? 0u : (rem >= 32 ? 0xFFFFFFFFu : ((1u << rem) - 1u));
            a.alive[1][w] = 0u;
            a.alive[2][w] = 0u;
        }
        for (long long k = tid; k < a.max_steps; k += nth) a.work[k] = 0;
        if (tid < 3) a.bar[tid * 32] = 0;  // arrivals, go word, abort flag (cd_step.cuh LB_*)
    }
    if (tid == 0) {
        if (a.n_active) *a.n_active = none ? 0 : B;
        a.ctrs[2] = 0;
    }
}

// cd_decode_loop_async on the per-step path: the loop's error count joins the status word the host reads in
// cd_loop_sync (pinned, device-mapped host memory).
__global__ void fold_status_kernel(const int* __restrict__ ctrs, int* host_status) {
    const int err = __ldcg(ctrs + 2);
    if (err) atomicAdd_system(host_status, err);
}

// Host-buffer loop (cd_decode_loop_host) when the caller's logits are in pinned, device-mapped host
// memory: the rows still active are pulled over PCIe by the SMs themselves, straight from the host
// buffer into the compact staging buffer (row = slot) -- no host read of the active list, no
// per-row copy calls.  16-byte loads, 4 independent ones per thread in flight.
__global__ void host_gather_rows_kernel(const unsigned char* __restrict__ src, unsigned long long row_bytes,
                                        const int* __restrict__ row_ids, const int* __restrict__ n_dev,
                                        unsigned char* __restrict__ dst) {
    const int n = __ldcg(n_dev);
    const unsigned long long vec_per_row = row_bytes >> 4;
    const unsigned long long total = (unsigned long long)n * vec_per_row;
    const unsigned long long nth = (unsigned long long)gridDim.x * blockDim.x;
    unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 3 * nth < total; i += 4 * nth) {
        uint4 v[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const unsigned long long j = i + q * nth;
            const unsigned long long slot = j / vec_per_row, off = j - slot * vec_per_row;
            v[q] = *reinterpret_cast<const uint4*>(src + (unsigned long long)__ldg(row_ids + slot) * row_bytes + (off << 4));
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const unsigned long long j = i + q * nth;
            reinterpret_cast<uint4*>(dst)[j] = v[q];
        }
    }
    for (; i < total; i += nth) {
        const unsigned long long slot = i / vec_per_row, off = i - slot * vec_per_row;
        reinterpret_cast<uint4*>(dst)[i] =
            *reinterpret_cast<const uint4*>(src + (unsigned long long)__ldg(row_ids + slot) * row_bytes + (off << 4));
    }
}

// Measurement aid (cd_probe_read): the copy machinery of the step kernel -- per-warp rings of 1-D bulk
// async copies on mbarriers, 12 warps x 2 stages x 8 KiB per SM -- streaming a buffer with NO arithmetic
// (one word per tile is read so the copy is not dead).  What it reaches is the ceiling of a pure-read
// kernel of this shape on this GPU.
template <int WARPS, int STAGES, int TILE>
__global__ void __launch_bounds__(WARPS * 32, 1) read_probe_kernel(const unsigned char* __restrict__ p,
                                                                   unsigned long long ntiles, unsigned* sink) {
    extern __shared__ __align__(128) unsigned char probe_smem[];
    __shared__ __align__(8) unsigned long long bars[WARPS * STAGES];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned char* ring = probe_smem + (size_t)warp * STAGES * TILE;
    unsigned long long* bar = bars + warp * STAGES;
    if (lane == 0) {
        for (int s = 0; s < STAGES; ++s) mbar_init(smem_u32(&bar[s]), 1);
        fence_mbar_init();
    }
    __syncwarp();
    const unsigned long long tw = (unsigned long long)gridDim.x * WARPS;
    unsigned long long next = (unsigned long long)blockIdx.x * WARPS + warp;
    int in_flight = 0, st_i = 0, st_c = 0;
    uint32_t phase = 0;
    unsigned acc = 0;
    auto issue = [&]() {
        if (next >= ntiles) return;
        if (lane == 0) {
            mbar_arrive_expect_tx(smem_u32(&bar[st_i]), TILE);
            bulk_g2s(smem_u32(ring + st_i * TILE), p + next * TILE, TILE, smem_u32(&bar[st_i]));
        }
        next += tw;
        ++in_flight;
        st_i = (st_i + 1 == STAGES) ? 0 : st_i + 1;
    };
    for (int s = 0; s < STAGES; ++s) issue();
    while (in_flight > 0) {
        mbar_wait(smem_u32(&bar[st_c]), phase);
        acc ^= reinterpret_cast<const unsigned*>(ring + st_c * TILE)[lane];
        --in_flight;
        st_c = (st_c + 1 == STAGES) ? 0 : st_c + 1;
        phase ^= (st_c == 0) ? 1u : 0u;
        __syncwarp();
        issue();
    }
    if (acc == 0x9E3779B9u && sink) *sink = acc;  // practically never: keeps the loads alive
}

}  // namespace cd
