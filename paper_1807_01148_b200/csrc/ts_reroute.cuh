// ts_reroute.cuh -- iterative decaying re-routing on the device.
//
// PAPER.md:386 (section 6.3.1): "After that first iteration, we use the microsimulation measurements to
// update those weights and repeat the microsimulation ... we recompute all routes the first and second
// iteration, and then we decay it to half and one-fourth of the vehicles"; PAPER.md:431 (section 6.3.5):
// per-vehicle Dijkstra is replaced by shortest paths for everybody at once.  Readings R37-R41 in
// integer edge weights in 1/256 step from the edge statistics the step kernels keep;
// one shortest-path tree per distinct origin node; ties settled by (distance, edge id).
//
// Kernels (product code, sm_100a; shares nothing with oracle/reroute.py):
//   k_rr_weights   w[e] = round-half-up(256 * exit_steps_sum / exited), else the caller's free-flow weight
//   k_rr_pack      per outbound edge in CSR order { edge id, head node, weight, where the head's records start }
//   k_rr_sssp      one CTA of 256 threads per origin node, 592 in flight: label-correcting shortest paths over the CSR of outbound
//                  edges, frontier by frontier; a node's label is ONE 64-bit word (distance << 32 |
//                  inbound edge) under atomicMin, so the lexicographic minimum IS the tie-break rule
//   k_rr_len       per vehicle: length of its new route (walk the tree back from the destination)
//   k_rr_scan*     exclusive scan of the lengths -> route offsets
//   k_rr_write     per vehicle: write the new route (or copy the old one) at its offset
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ts {

constexpr uint32_t kRrNone = 0xFFFFFFFFu;
constexpr uint32_t kRrUnit = 256;            // weight units per simulation step (R37)
constexpr uint32_t kRrWMax = 1u << 20;
// Shortest-path trees in flight, one CTA of kRrThreads threads each.  A frontier of a road network holds a few
// hundred nodes and a tree is a chain of ~diameter frontiers, each a __syncthreads() apart: small CTAs, many of them
// (4 per SM), finish 4 096 trees of config 3 four times sooner than one 1 024-thread CTA per SM did.
constexpr uint32_t kRrCtas = 592, kRrThreads = 256;

struct RrCtx {
    uint32_t V, E, N, n_src;
    // graph
    const uint32_t* out_off;       // [N+1] CSR by tail node
    const uint32_t* out_edge;      // [E]   edge ids, ascending inside a node
    const uint32_t* edge_from;     // [E]
    const uint32_t* edge_to;       // [E]
    uint32_t* w;                   // [E]   routing weights of this call
    uint4* adjw;                   // [E+4] by CSR position: one record per outbound edge (k_rr_pack)
    const uint32_t* w_free;        // [E]   the caller's free-flow weights
    // measurements (the step kernels' accumulators)
    const uint32_t* st_exited;
    const unsigned long long* st_exit_steps;
    // demand
    const uint32_t* origin;        // [V] tail node of the first route edge (never changes)
    const uint32_t* dest;          // [V] head node of the last route edge (never changes)
    const uint32_t* src_idx;       // [V] index of the origin in src_node
    const uint32_t* src_node;      // [n_src]
    const uint8_t* mask;           // [V] re-route this vehicle
    const uint32_t* old_routes;    // route table in use
    const uint32_t* old_begin;     // [V]
    const uint32_t* old_end;       // [V]
    uint32_t* new_routes;          // the other route table
    uint32_t* new_len;             // [V+1]
    uint32_t* new_off;             // [V+1] exclusive scan of new_len
    uint32_t* block_sum;           // scan scratch
    uint32_t* first2;              // [2V] first and second edge of every new route (for the host's queue index)
    // trees
    uint32_t* pred;                // [n_src][N] inbound edge on the shortest path from the source, kRrNone = none
    unsigned long long* lab;       // [kRrCtas][N] labels of the trees in flight
    uint2* fa; uint2* fb;          // [kRrCtas][N] frontiers: { node, CSR position of its first outbound edge }
    uint32_t* stamp;               // [kRrCtas][N] last frontier a node was put in
    uint32_t* error;               // sticky: 1 = a path cost passed 2^32
};

__global__ void k_rr_weights(const RrCtx r) {
    for (uint32_t e = blockIdx.x * blockDim.x + threadIdx.x; e < r.E; e += gridDim.x * blockDim.x) {
        const unsigned long long n = r.st_exited[e];
        unsigned long long w = r.w_free[e];
        if (n) w = (r.st_exit_steps[e] * kRrUnit + n / 2) / n;
        w = w < 1 ? 1 : (w > kRrWMax ? kRrWMax : w);
        r.w[e] = (uint32_t)w;
    }
}

// What a relaxation needs of an outbound edge, side by side in CSR order -- one 16-byte record instead of the edge id
// followed by its head node and weight:
//   { edge id | kRrLast on the last outbound edge of its tail node, head node, weight of this call,
//     CSR position of the HEAD node's first outbound edge (kRrNone if it has none) }
// The last word lets a frontier entry carry where its node's records start, so that a node's label and its records
// are fetched in the same trip.  Edge ids stay below 2^31.  Run before every k_rr_sssp.
constexpr uint32_t kRrLast = 0x80000000u;
__global__ void k_rr_pack(const RrCtx r) {
    for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < r.E; j += gridDim.x * blockDim.x) {
        const uint32_t e = r.out_edge[j], u = r.edge_from[e], v = r.edge_to[e];
        const uint32_t hv = r.out_off[v] < r.out_off[v + 1] ? r.out_off[v] : kRrNone;
        r.adjw[j] = make_uint4(e | (j + 1 == r.out_off[u + 1] ? kRrLast : 0u), v, r.w[e], hv);
    }
}

// todo[0..n_todo): indices into src_node of the trees wanted.
// Frontier entries are { node, CSR position of its first outbound edge }; fa / fb hold N of them per tree in flight.
__global__ void __launch_bounds__(kRrThreads) k_rr_sssp(const RrCtx r, const uint32_t* __restrict__ todo, uint32_t n_todo) {
    __shared__ uint32_t sh_next;
    const uint32_t t = threadIdx.x, T = blockDim.x, N = r.N;
    unsigned long long* lab = r.lab + (size_t)blockIdx.x * N;
    uint32_t* stamp = r.stamp + (size_t)blockIdx.x * N;
    uint2* fa = r.fa + (size_t)blockIdx.x * N;
    uint2* fb = r.fb + (size_t)blockIdx.x * N;
    for (uint32_t si = blockIdx.x; si < n_todo; si += gridDim.x) {
        const uint32_t s_idx = todo[si], s = r.src_node[s_idx];
        for (uint32_t v = t; v < N; v += T) { lab[v] = ~0ull; stamp[v] = 0u; }
        __syncthreads();
        const uint32_t s_first = r.out_off[s] < r.out_off[s + 1] ? r.out_off[s] : kRrNone;
        if (t == 0) { lab[s] = (unsigned long long)kRrNone; fa[0] = make_uint2(s, s_first); sh_next = 0; }   // distance 0, no inbound edge
        __syncthreads();
        uint32_t n_f = s_first != kRrNone ? 1u : 0u, epoch = 0;
        while (n_f) {
            epoch++;
            for (uint32_t i = t; i < n_f; i += T) {
                const uint2 ent = __ldcg(fa + i);
                // The outbound edges of the node four at a time, every load of a stage issued before any is
                // consumed: a frontier is a chain of dependent trips to L2 (entry -> label and edge records ->
                // atomicMin -> stamp), and edge after edge they were what a tree took (a node of a road network has
                // 3-4 outbound edges).  Same labels at the end: the minimum does not depend on the order of the
                // attempts.  Records read beyond the node's last one are ignored (adjw has 4 spare records).
                const unsigned long long du = __ldcg(lab + ent.x) >> 32;
                bool more = true;
                for (uint32_t j = ent.y; more; j += 4) {
                    uint4 a[4];
                    unsigned long long cand[4], old[4];
                    bool go[4];
#pragma unroll
                    for (int q = 0; q < 4; q++) a[q] = r.adjw[j + q];
#pragma unroll
                    for (int q = 0; q < 4; q++) {
                        go[q] = more;
                        if (a[q].x & kRrLast) more = false;
                        const unsigned long long nd = du + a[q].z;
                        if (go[q] && nd >= 0xFFFFFFFFull) { *r.error = 1u; go[q] = false; }
                        cand[q] = (nd << 32) | (a[q].x & ~kRrLast);
                    }
#pragma unroll
                    for (int q = 0; q < 4; q++) if (go[q]) old[q] = atomicMin(lab + a[q].y, cand[q]);
                    // a shorter distance: v's outbound edges must be relaxed again.  (The same distance over
                    // a lower edge id only replaces the inbound edge.)  A head node without outbound edges has
                    // nothing to relax and stays out of the frontier.
                    uint32_t seen[4];
#pragma unroll
                    for (int q = 0; q < 4; q++) {
                        go[q] = go[q] && cand[q] < old[q] && (cand[q] >> 32) < (old[q] >> 32) && a[q].w != kRrNone;
                        if (go[q]) seen[q] = atomicExch(stamp + a[q].y, epoch);
                    }
#pragma unroll
                    for (int q = 0; q < 4; q++) if (go[q] && seen[q] != epoch) fb[atomicAdd(&sh_next, 1u)] = make_uint2(a[q].y, a[q].w);
                }
            }
            __syncthreads();
            n_f = sh_next;
            __syncthreads();
            if (t == 0) sh_next = 0;
            uint2* tmp = fa; fa = fb; fb = tmp;
            __threadfence_block();
            __syncthreads();
        }
        uint32_t* row = r.pred + (size_t)s_idx * N;
        for (uint32_t v = t; v < N; v += T) row[v] = (uint32_t)__ldcg(lab + v);
        __syncthreads();
    }
}

// A vehicle's new route: R39 (mask), R40 (origin == destination or unreachable: keeps its route).
__device__ __forceinline__ bool rr_wants(const RrCtx& r, uint32_t i, const uint32_t*& row) {
    if (!r.mask[i]) return false;
    const uint32_t o = r.origin[i], d = r.dest[i];
    row = r.pred + (size_t)r.src_idx[i] * r.N;
    return o != d && row[d] != kRrNone;
}

__global__ void k_rr_len(const RrCtx r) {
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < r.V; i += gridDim.x * blockDim.x) {
        const uint32_t* row;
        uint32_t n = r.old_end[i] - r.old_begin[i];
        if (rr_wants(r, i, row)) {
            const uint32_t o = r.origin[i];
            uint32_t v = r.dest[i];
            for (n = 0; v != o && n <= r.N; n++) v = r.edge_from[row[v]];
        }
        r.new_len[i] = n;
    }
}

// exclusive scan of new_len[0..V] (V+1 items, the last one a zero) in three passes; totals < 2^32
constexpr uint32_t kScanBlock = 256, kScanItems = 8;
__global__ void __launch_bounds__(kScanBlock) k_rr_scan1(const uint32_t* in, uint32_t* out, uint32_t* block_sum, uint32_t n) {
    __shared__ uint32_t sh[kScanBlock];
    const uint32_t base = (blockIdx.x * kScanBlock + threadIdx.x) * kScanItems;
    uint32_t v[kScanItems], s = 0;
    for (uint32_t j = 0; j < kScanItems; j++) { v[j] = base + j < n ? in[base + j] : 0u; s += v[j]; }
    sh[threadIdx.x] = s;
    __syncthreads();
    for (uint32_t o = 1; o < kScanBlock; o <<= 1) {
        const uint32_t a = threadIdx.x >= o ? sh[threadIdx.x - o] : 0u;
        __syncthreads();
        sh[threadIdx.x] += a;
        __syncthreads();
    }
    uint32_t run = sh[threadIdx.x] - s;
    for (uint32_t j = 0; j < kScanItems; j++) { if (base + j < n) out[base + j] = run; run += v[j]; }
    if (threadIdx.x == kScanBlock - 1) block_sum[blockIdx.x] = sh[threadIdx.x];
}
__global__ void k_rr_scan2(uint32_t* block_sum, uint32_t n_blocks) {       // one thread: n_blocks is a few thousand
    if (blockIdx.x || threadIdx.x) return;
    uint32_t run = 0;
    for (uint32_t b = 0; b < n_blocks; b++) { const uint32_t s = block_sum[b]; block_sum[b] = run; run += s; }
}
__global__ void __launch_bounds__(kScanBlock) k_rr_scan3(uint32_t* out, const uint32_t* block_sum, uint32_t n) {
    const uint32_t base = (blockIdx.x * kScanBlock + threadIdx.x) * kScanItems, add = block_sum[blockIdx.x];
    for (uint32_t j = 0; j < kScanItems; j++) if (base + j < n) out[base + j] += add;
}

__global__ void k_rr_write(const RrCtx r) {
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < r.V; i += gridDim.x * blockDim.x) {
        const uint32_t* row;
        const uint32_t off = r.new_off[i], n = r.new_len[i];
        if (rr_wants(r, i, row)) {
            const uint32_t o = r.origin[i];
            uint32_t v = r.dest[i];
            for (uint32_t j = n; j-- > 0 && v != o;) { const uint32_t e = row[v]; r.new_routes[off + j] = e; v = r.edge_from[e]; }
        } else {
            const uint32_t b = r.old_begin[i];
            for (uint32_t j = 0; j < n; j++) r.new_routes[off + j] = r.old_routes[b + j];
        }
    }
}
// first and second edge of every route (the host rebuilds the departure-queue index from them)
__global__ void k_rr_first2(const RrCtx r) {
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < r.V; i += gridDim.x * blockDim.x) {
        const uint32_t off = r.new_off[i], n = r.new_len[i];
        r.first2[2 * (size_t)i] = r.new_routes[off];
        r.first2[2 * (size_t)i + 1] = n > 1 ? r.new_routes[off + 1] : kRrNone;
    }
}

}  // namespace ts
