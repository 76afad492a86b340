// ts_sort.cuh -- compaction of retired slots and re-sort of the live ones by edge (SURVEY.md
// 8(a) rows A9 and A10; BASELINE.json "a warp-scan compaction of departing and arriving vehicles,
// and a periodic re-sort of vehicles by edge for locality").
//
// One counting sort does both, in four grid-wide passes over the slots / the edge table:
//   sort_rank    : every live slot takes a rank among the vehicles of its edge (integer atomicAdd
//                  on the edge histogram); retired slots get none -- that is the compaction
//   sort_partial : each CTA sums its contiguous share of the histogram (warp shuffles)
//   sort_scan    : exclusive scan of the histogram: CTA offset from the partial sums, then a
//                  block-wide warp-scan over the CTA's share; the histogram is zeroed for next time
//   sort_scatter : live slots move to base[edge] + rank in the other slot set
// The order of vehicles inside one edge depends on atomic arrival order and is NOT reproducible;
// nothing the simulation computes depends on slot order (arbitration is by vehicle id), which is
// what the parity tests with different sort periods check.
#pragma once
#include "ts_device.cuh"

namespace ts {

__device__ __forceinline__ uint32_t warp_sum(uint32_t v) {
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    return v;
}
__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v) {
    const uint32_t lane = threadIdx.x & 31u;
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t n = __shfl_up_sync(0xFFFFFFFFu, v, o);
        if (lane >= (uint32_t)o) v += n;
    }
    return v;
}
// Block-wide sum; `red` is 33 words of shared memory.  Every thread gets the result.
__device__ __forceinline__ uint32_t block_sum(uint32_t v, uint32_t* red) {
    const uint32_t w = threadIdx.x >> 5, lane = threadIdx.x & 31u, nw = (blockDim.x + 31u) >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) red[w] = v;
    __syncthreads();
    if (w == 0) {
        uint32_t s = lane < nw ? red[lane] : 0u;
        s = warp_sum(s);
        if (lane == 0) red[32] = s;
    }
    __syncthreads();
    return red[32];
}

// Sort key: the edge, and above it the vehicle's place in the lane-change stagger (readings
// R10/R14: vehicle id takes its turn when ((k >> 1) + id) % lc_period == 0), so that the warps of
// one group evaluate lane changes together and the others skip that code.
__device__ __forceinline__ uint32_t sort_key(const Ctx& c, const uint4& sb) {
    return (sb.z & (c.sort_groups - 1u)) * c.E + sb.x;
}

__device__ __forceinline__ uint32_t sort_rank(const Ctx& c, const Slots& S, const Who& me, uint32_t n) {
    for (uint32_t j = 0;; j++) {
        const uint32_t s = me.slot(j);
        if (s >= n) break;
        const uint4 sa = ldcg4(S.A + s);
        uint32_t r = NONE32;
        if (sa.w & ALIVE) {
            const uint4 sb = ldcg4(S.B + s);
            r = atomicAdd(c.hist + sort_key(c, sb), 1u);
        }
        c.rank[s] = r;
    }
    // a slot reserved by a waiting departure is not alive and goes away with this compaction
    for (uint32_t q = me.gtid(); q < c.n_queues; q += me.gthreads()) c.queue_state[q].z = NONE32;
    return n;
}

__device__ __forceinline__ uint32_t n_keys(const Ctx& c) { return c.sort_groups * c.E; }
__device__ __forceinline__ uint32_t edge_share(const Ctx& c, const Who& me) { return (n_keys(c) + me.n_cta - 1) / me.n_cta; }

__device__ __forceinline__ void sort_partial(const Ctx& c, const Who& me, uint32_t* red) {
    const uint32_t share = edge_share(c, me), lo = me.cta * share, hi = min(n_keys(c), lo + share);
    uint32_t s = 0;
    for (uint32_t e = lo + me.t; e < hi; e += me.T) s += __ldcg(c.hist + e);
    s = block_sum(s, red);
    if (me.t == 0) c.partial[me.cta] = s;
}

__device__ __forceinline__ void sort_scan(const Ctx& c, const Who& me, uint32_t* red) {
    const uint32_t share = edge_share(c, me), lo = me.cta * share, hi = min(n_keys(c), lo + share);
    uint32_t mine = 0;
    for (uint32_t b = me.t; b < me.cta; b += me.T) mine += __ldcg(c.partial + b);
    uint32_t run = block_sum(mine, red);                                    // exclusive offset of this CTA
    const uint32_t w = me.t >> 5, lane = me.t & 31u, nw = (me.T + 31u) >> 5;
    for (uint32_t e0 = lo; e0 < hi; e0 += me.T) {
        const uint32_t e = e0 + me.t;
        const uint32_t h = e < hi ? __ldcg(c.hist + e) : 0u;
        const uint32_t inc = warp_incl_scan(h);
        __syncthreads();
        if (lane == 31) red[w] = inc;
        __syncthreads();
        if (w == 0) {
            const uint32_t ws = lane < nw ? red[lane] : 0u;
            const uint32_t wi = warp_incl_scan(ws);
            red[lane] = wi - ws;                                            // exclusive offset of warp `lane`
            if (lane == 31) red[32] = wi;                                   // tile total
        }
        __syncthreads();
        if (e < hi) { c.base[e] = run + red[w] + inc - h; c.hist[e] = 0u; }
        run += red[32];
    }
    if (me.cta == me.n_cta - 1 && me.t == 0) {                              // run == number of live slots
        c.dyn->slot_alloc = run;
        c.dyn->n_slots = run;
    }
}

__device__ __forceinline__ void sort_scatter(const Ctx& c, const Slots& from, const Slots& to, const Who& me, uint32_t n) {
    for (uint32_t j = 0;; j++) {
        const uint32_t s = me.slot(j);
        if (s >= n) break;
        const uint32_t r = __ldcg(c.rank + s);
        if (r == NONE32) continue;
        const uint4 sa = ldcg4(from.A + s), sb = ldcg4(from.B + s), sc = ldcg4(from.C + s);
        const uint32_t d = __ldcg(c.base + sort_key(c, sb)) + r;
        stcg4(to.A + d, sa); stcg4(to.B + d, sb); stcg4(to.C + d, sc);
        if (from.D) __stcg(to.D + d, __ldcg(from.D + s));
    }
}

}  // namespace ts
