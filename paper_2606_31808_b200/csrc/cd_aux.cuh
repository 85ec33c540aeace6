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

// a6 as a kernel of its own (cd_compact): one CTA of 1024 threads, see block_compact.
__global__ void __launch_bounds__(1024, 1) compact_kernel(const uint8_t* done, const int* row_ids_in,
                                                          const int* state_in, int n, int* row_ids_out,
                                                          int* state_out, int* n_active_out) {
    block_compact(done, row_ids_in, state_in, n, row_ids_out, state_out, n_active_out);
}

// a7 set-up: every row starts in the start state with an empty history.
__global__ void loop_init_kernel(int B, int max_steps, int start, int start_accepting, int* row_ids,
                                 int* state, int* n_active, int* tokens_out, int* len_out,
                                 int* final_state_out, float* sum_logprob_out, uint8_t* done_row_out,
                                 const int* sat_ctr, int limit) {
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
    // LIMIT already satisfied by earlier batches: no row takes a step
    if (tid == 0) *n_active = (start_accepting || (sat_ctr && *sat_ctr >= limit)) ? 0 : B;
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
