// cd_dedup.cuh -- early deduplication and cascade filtering as device primitives (
// PAPER.md section 2.4 "Early Deduplication of Database Values", L156, and "Cascade Filtering",
// L150).  Row values are 64-bit keys (interned value ids or hashes of the column values):
//   dedup_insert_kernel   SELECT DISTINCT: open-addressing hash table, one 64-bit CAS to claim a
//                         slot + atomicMin of the row id, so every distinct value knows its FIRST row
//   dedup_first_kernel    every row looks its value up: first[i] = first row with the same value
//   (ranking)             the stable compaction of a6 over the rows that are first occurrences
//                         (cd_aux.cuh compact_lookback_kernel: many CTAs, decoupled look-back) ->
//                         distinct_rows[] (ascending row id = first-occurrence order) and the rank
//                         of each of them
//   dedup_rep_kernel      rep[i] = rank[first[i]]   (the key of the LEFT JOIN back)
//   join_kernel           LEFT JOIN: broadcast the distinct rows' decode results to all rows
//   filter_kernel         cascade: rows that finished in a satisfying state, in row order
#pragma once
#include "cd_common.cuh"

namespace cd {

constexpr unsigned long long DEDUP_EMPTY = 0x8000000000000000ull;  // INT64_MIN marks a free slot

__device__ __forceinline__ uint32_t dedup_hash(unsigned long long k, uint32_t mask) {
    k ^= k >> 33;
    k *= 0xff51afd7ed558ccdull;
    k ^= k >> 33;
    k *= 0xc4ceb9fe1a85ec53ull;
    k ^= k >> 33;
    return (uint32_t)k & mask;
}

__global__ void dedup_clear_kernel(unsigned long long* tkey, long long n) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        tkey[i] = DEDUP_EMPTY;
}

// table: cap slots of {key, min row}; cap is a power of two >= 2N; slot `cap` is reserved for the
// key INT64_MIN itself.  Pre-set: keys = DEDUP_EMPTY, minrow = INT_MAX.
__global__ void dedup_insert_kernel(const long long* __restrict__ keys, int N, unsigned long long* tkey,
                                    int* tmin, uint32_t cap) {
    const uint32_t mask = cap - 1u;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        const unsigned long long k = (unsigned long long)keys[i];
        uint32_t slot;
        if (k == DEDUP_EMPTY) {
            slot = cap;
        } else {
            slot = dedup_hash(k, mask);
            while (true) {
                const unsigned long long cur = atomicCAS(tkey + slot, DEDUP_EMPTY, k);
                if (cur == DEDUP_EMPTY || cur == k) break;
                slot = (slot + 1u) & mask;
            }
        }
        atomicMin(tmin + slot, (int)i);
    }
}

__global__ void dedup_first_kernel(const long long* __restrict__ keys, int N, const unsigned long long* __restrict__ tkey,
                                   const int* __restrict__ tmin, uint32_t cap, int* __restrict__ first,
                                   uint8_t* __restrict__ not_first) {
    const uint32_t mask = cap - 1u;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        const unsigned long long k = (unsigned long long)keys[i];
        uint32_t slot;
        if (k == DEDUP_EMPTY) {
            slot = cap;
        } else {
            slot = dedup_hash(k, mask);
            while (tkey[slot] != k) slot = (slot + 1u) & mask;
        }
        const int f = tmin[slot];
        first[i] = f;
        not_first[i] = (f == (int)i) ? 0 : 1;
    }
}

__global__ void dedup_rep_kernel(const int* __restrict__ first, const int* __restrict__ rank, int N, int* __restrict__ rep) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x)
        rep[i] = rank[first[i]];
}

// LEFT JOIN back: row i receives the decode results of distinct value rep[i].
__global__ void join_kernel(const int* __restrict__ rep, int N, int max_steps, const int* __restrict__ tokens_d,
                            const int* __restrict__ len_d, const int* __restrict__ fs_d, const float* __restrict__ slp_d,
                            const uint8_t* __restrict__ done_d, int* __restrict__ tokens, int* __restrict__ len,
                            int* __restrict__ fs, float* __restrict__ slp, uint8_t* __restrict__ done, int vec_lanes) {
    const long long nth = (long long)gridDim.x * blockDim.x;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (vec_lanes > 0) {
        // token rows of whole 16-byte vectors (max_steps % 4 == 0, both arrays 16-byte aligned): a group of vec_lanes
        // lanes (a power of two <= 32) per row -- rep[i] is read once per row (one broadcast load per group), the
        // history moves as int4, the group's first lane carries the row's scalar results
        const int vpr = max_steps >> 2;
        const int sub = (int)(tid & (vec_lanes - 1));
        const int sh = __ffs(vec_lanes) - 1;  // (no 64-bit division on the index path)
        for (long long i = tid >> sh; i < N; i += nth >> sh) {
            const int r = rep[i];
            if (sub == 0) {
                if (len) len[i] = len_d[r];
                if (fs) fs[i] = fs_d[r];
                if (slp) slp[i] = slp_d[r];
                if (done) done[i] = done_d[r];
            }
            const int4* __restrict__ src = reinterpret_cast<const int4*>(tokens_d + (long long)r * max_steps);
            int4* __restrict__ dst = reinterpret_cast<int4*>(tokens + i * max_steps);
            for (int k = sub; k < vpr; k += vec_lanes) dst[k] = __ldg(src + k);
        }
        return;
    }
    for (long long i = tid; i < N; i += nth) {
        const int r = rep[i];
        if (len) len[i] = len_d[r];
        if (fs) fs[i] = fs_d[r];
        if (slp) slp[i] = slp_d[r];
        if (done) done[i] = done_d[r];
    }
    if (tokens) {
        // one warp per row: coalesced over the steps, no division per element
        const int lane = threadIdx.x & 31;
        for (long long i = tid >> 5; i < N; i += nth >> 5) {
            const long long src = (long long)rep[i] * max_steps, dst = i * max_steps;
            for (int k = lane; k < max_steps; k += 32) tokens[dst + k] = tokens_d[src + k];
        }
    }
}

// Cascade filtering: flag = 1 for rows that are NOT passed on to the next LM
// predicate (did not finish, or finished in a state outside the satisfying set).
__global__ void filter_flag_kernel(const int* __restrict__ final_state, const uint8_t* __restrict__ done, int N,
                                   const uint8_t* __restrict__ satisfying, int S, uint8_t* __restrict__ drop) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        const int s = final_state[i];
        drop[i] = (done[i] && s >= 0 && s < S && satisfying[s]) ? 0 : 1;
    }
}

}  // namespace cd
