// ts_device.cuh -- device-side data layout and helpers of the traffic microsimulation
// (sections 6.3.2-6.3.3; rule set in DESIGN.md section 2).
//
// Product code for sm_100a.  Shares nothing with oracle/.  Built with -fmad=false and IEEE
// division so that every fp32 expression below is the written sequence of single operations.
//
// One simulation step k -> k+1 is two grid-wide phases (ts_phases.cuh):
//   phase 1 : every ACTIVE vehicle reads its own state k and the traffic atlas M_k, decides lane
//             change / acceleration / crossing, WRITES ITS OWN STATE k+1 (nobody else reads it) and
//             leaves a 16-byte move record; crossing vehicles and ready departure-queue heads post
//             step-tagged atomicMin claims (lowest vehicle id wins).
//   -- grid-wide dependency: every scan of M_k done, every claim visible --
//   phase 2 : move records are applied to the atlas (old cell vacated, new cell occupied: single
//             buffer, race-free by invariant I6); the few crossing vehicles and departures resolve
//             their claims and commit.
//   -- grid-wide dependency: M_{k+1} complete --
// Every R steps the slots are compacted and re-sorted by edge (ts_sort.cuh); results never depend
// on slot order because arbitration keys are vehicle ids.
//
// The traffic atlas is two planes over the same rows.  A lane row is
// `stride` chunks of 128 cells (one cell = one metre), zero-padded:
//   code plane : one byte per cell, the occupant's speed code (valid only where occupied);
//   occupancy  : one bit per cell, 16 bytes per chunk, so that "check the following bytes" for a
//                128-cell lookahead is two independent 16-byte loads and an __ffs instead of a
//                chain of up to nine dependent loads.
// Vacating a cell clears its bit only; stale code bytes are never read.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ts {

constexpr uint32_t NONE32 = 0xFFFFFFFFu;
enum : uint32_t { CTRL_FREE = 0, CTRL_PRIORITY = 1, CTRL_SIGNAL = 2 };
enum : uint32_t { ERR_CELL_CLASH = 1, ERR_SLOTS = 2, ERR_LOGIC = 4 };
enum : uint32_t { ALIVE = 0x100u };
// move-record kinds (uint4.w)
enum : uint32_t { MR_NONE = 0, MR_MOVE = 1, MR_CLEAR = 2, MR_CROSS = 3 };

// 32 bytes per edge: everything a vehicle needs to know about the edge it is on (or enters),
// including the signal plan of the node at its head, in two 16-byte loads.
struct __align__(16) EdgeRec {
    uint32_t row;        // atlas offset of lane 0's row, in chunks of 128 cells
    uint32_t lane_base;  // global lane index of lane 0 (index of its claim word)
    float vlim;          // m/s
    uint32_t to_node;
    uint32_t cycle;      // n_in * (green + allred) at a SIGNAL head node, else 1
    uint32_t offset;     // signal offset, steps
    uint16_t green, P;   // P = green + allred
    uint16_t len;        // cells
    uint8_t lanes_ctrl;  // lanes | ctrl << 4
    uint8_t in_rank;     // rank among the inbound edges of the head node
};
static_assert(sizeof(EdgeRec) == 32, "EdgeRec must be 32 bytes");

// Counters that change during a run; one cache line in device memory.
struct Dyn {
    uint32_t n_departed, n_arrived;
    uint32_t slot_alloc;   // slots handed out so far (departures append here)
    uint32_t n_slots;      // slots visible to the step in flight
    uint32_t error;        // sticky ERR_*
    uint32_t n_samples;
    uint32_t k;            // step counter
    uint32_t pad;
    unsigned long long sum_arrive, updates;
};

struct Params {
    float dt, a, b, T, s0, len, b_safe, politeness, lc_threshold;
    float K;               // 2*sqrtf(a*b), computed once on the host in fp32
    float half_a_dt;       // (0.5f*a)*dt   (E4)
    float a_dt;            // a*dt          (E5)
    float entry_zone_f;
    int H, Hb;
    uint32_t lc_period, insert_clear, sample_period;
};

// Slot-ordered vehicle state: three 16-byte vectors per slot (two ping-pong sets, swapped by
// the re-sort).
//   A = { bits(x), bits(v), row (first chunk of the vehicle's lane row), lane | ALIVE }
//   B = { edge, next route edge or NONE32, vehicle id, bits(v0_mult) }
//   C = { route position, one past the last route position, step it entered the edge, bits(mand_dist) }
struct Slots {
    uint4* A;
    uint4* B;
    uint4* C;
};

// Everything the kernels touch.  Passed by value.
struct Ctx {
    Params p;
    uint32_t V, E, N, n_queues, cap_slots;
    // static network / demand
    const EdgeRec* edges;               // [E]
    const uint32_t* route_edges;        // [R]
    const uint32_t* route_begin;        // [V] first position of the vehicle's route
    const uint4* queue_rec;             // [Q] { row of lane 0, lane_base, end position, edge }
    const uint4* dep_rec;               // [2V] by queue position: { id, v0_mult, mand, rbegin } { rend, next, dep_step, 0 }
    // mutable
    uint8_t* codes;                     // traffic atlas, code plane: one byte per metre of lane
    uint4* occ;                         // traffic atlas, occupancy plane: one bit per metre
    uint4* queue_state;                 // [Q] { head position, departure step of the head, reserved slot or NONE32, - }
    uint4* queue_cand;                  // [Q] { candidate id or NONE32, its slot, head, dep step of the next }
    unsigned long long* lane_claim;     // [n_lanes] step-tagged minimum id
    unsigned long long* node_claim;     // [N]
    Dyn* dyn;
    unsigned int* barrier;              // grid barrier counter of the persistent kernel
    Slots s[2];
    uint4* mr_g;                        // [cap] move records that do not fit in shared memory
    uint4* cr;                          // [2 cap] crossing records
    // compaction + re-sort scratch
    uint32_t* rank;                     // [cap]
    uint32_t* hist;                     // [E]
    uint32_t* base;                     // [E]
    uint32_t* partial;                  // [kMaxCtas]
    // id-ordered results
    uint8_t* o_status; uint8_t* o_lane; uint32_t* o_edge; float* o_x; float* o_v;
    uint32_t* o_rpos; uint32_t* o_insert; uint32_t* o_arrive;
    // per-edge statistics
    uint32_t* st_entered; uint32_t* st_exited; unsigned long long* st_exit_steps;
    uint32_t* st_samp_cnt; unsigned long long* st_samp_code;
};

constexpr uint32_t kMaxCtas = 2048;

// Who am I in the grid: slots are dealt to CTAs in tiles of blockDim.x consecutive slots, round
// robin, so that consecutive (edge-sorted) slots sit in consecutive lanes of one warp.
struct Who {
    uint32_t t, T, cta, n_cta;
    __device__ __forceinline__ uint32_t slot(uint32_t j) const { return (j * n_cta + cta) * T + t; }
    __device__ __forceinline__ uint32_t gtid() const { return cta * T + t; }
    __device__ __forceinline__ uint32_t gthreads() const { return n_cta * T; }
};

// ------------------------------------------------------------------ small helpers

__device__ __forceinline__ uint32_t speed_code(float v) {
    float q = v * 4.0f;
    q = q + 0.5f;
    int c = (int)q;
    c = c > 254 ? 254 : c;
    return (uint32_t)(1 + c);
}
__device__ __forceinline__ float speed_decode(uint32_t code) { return (float)((int)code - 1) * 0.25f; }

// Eq. 7: a*(1 - (v/v0)^4 - (s*/s)^2), s* = s0 + max(0, vT + v dv / (2 sqrt(ab))).
__device__ __forceinline__ float idm_free(float v, float v0) {
    float r = v / v0;
    float r2 = r * r;
    float r4 = r2 * r2;
    return 1.0f - r4;
}
__device__ __forceinline__ float idm(const Params& p, float v, float v0, bool has, float s, float dv) {
    float fr = idm_free(v, v0);
    if (!has) return p.a * fr;
    float t = v * p.T;
    float u = v * dv;
    float w = u / p.K;
    t = t + w;
    t = fmaxf(t, 0.0f);
    float ss = p.s0 + t;
    float se = fmaxf(s, 0.5f);
    float q = ss / se;
    float q2 = q * q;
    float d = fr - q2;
    return p.a * d;
}

__device__ __forceinline__ bool signal_green(const EdgeRec& e, uint32_t k) {
    uint32_t t = (k + e.offset) % e.cycle;          // k, offset < 2^31
    uint32_t ph = t / e.P;
    return ph == e.in_rank && (t - ph * e.P) < e.green;
}

__device__ __forceinline__ EdgeRec load_edge(const EdgeRec* edges, uint32_t e) {
    const uint4* p = reinterpret_cast<const uint4*>(edges + e);
    uint4 a = __ldg(p), b = __ldg(p + 1);
    EdgeRec r;
    uint4* q = reinterpret_cast<uint4*>(&r);
    q[0] = a; q[1] = b;
    return r;
}
__device__ __forceinline__ uint32_t edge_lanes(const EdgeRec& e) { return e.lanes_ctrl & 15u; }
__device__ __forceinline__ uint32_t edge_ctrl(const EdgeRec& e) { return e.lanes_ctrl >> 4; }
__device__ __forceinline__ uint32_t row_stride(const EdgeRec& e) { return ((uint32_t)e.len + 127u) >> 7; }
__device__ __forceinline__ uint32_t lane_row(const EdgeRec& e, uint32_t lane) { return e.row + lane * row_stride(e); }

__device__ __forceinline__ unsigned long long claim_word(uint32_t k, uint32_t id) {
    // newer steps compare smaller, so a stale word never beats a live claim and nothing is cleared
    return ((unsigned long long)(0xFFFFFFFFu - k) << 32) | id;
}

// ---- occupancy windows: 256 cells = two 16-byte chunks of one lane row, loaded together ----
struct Win {
    uint4 a, b;   // chunk ch and chunk ch+1
    int base;     // cell index of bit 0 of a
};
// `row` = first chunk of the lane row, `ch` = first chunk wanted.  Both loads are unconditional:
// chunk ch+1 may belong to the next row (the plane ends with two spare chunks), callers mask by
// the last cell of the edge, so no clamping -- and no dependence on the edge record -- is needed.
__device__ __forceinline__ Win load_win(const uint4* occ, uint32_t row, int ch) {
    Win w;
    w.base = ch << 7;
    w.a = __ldcg(occ + row + ch);
    w.b = __ldcg(occ + row + ch + 1);
    return w;
}
__device__ __forceinline__ uint32_t win_word(const Win& w, int i) {
    switch (i) {
        case 0: return w.a.x; case 1: return w.a.y; case 2: return w.a.z; case 3: return w.a.w;
        case 4: return w.b.x; case 5: return w.b.y; case 6: return w.b.z; default: return w.b.w;
    }
}
// "we check the following bytes in memory": first occupied cell in [from, to]
// (inclusive, cells of the window), or -1.
__device__ __forceinline__ int first_occupied(const Win& w, int from, int to) {
    const int f = from - w.base, t = to - w.base;      // bit indices in [0, 256)
    if (f > t) return -1;
#pragma unroll
    for (int i = 0; i < 8; i++) {
        const int lo = i << 5;
        uint32_t m = win_word(w, i);
        if (f > lo) m &= (f - lo >= 32) ? 0u : (0xFFFFFFFFu << (f - lo));
        if (t < lo + 31) m &= (t < lo) ? 0u : (0xFFFFFFFFu >> (lo + 31 - t));
        if (m) return w.base + lo + __ffs((int)m) - 1;
    }
    return -1;
}
// Last occupied cell in [from, to] (the lag vehicle), or -1.
__device__ __forceinline__ int last_occupied(const Win& w, int from, int to) {
    const int f = from - w.base, t = to - w.base;
    if (f > t) return -1;
#pragma unroll
    for (int i = 7; i >= 0; i--) {
        const int lo = i << 5;
        uint32_t m = win_word(w, i);
        if (f > lo) m &= (f - lo >= 32) ? 0u : (0xFFFFFFFFu << (f - lo));
        if (t < lo + 31) m &= (t < lo) ? 0u : (0xFFFFFFFFu >> (lo + 31 - t));
        if (m) return w.base + lo + 31 - __clz((int)m);
    }
    return -1;
}
// General ranges (lookahead > 128 cells): window after window.
__device__ __forceinline__ int scan_ahead(const uint4* occ, uint32_t row, int from, int to) {
    if (from > to) return -1;
    for (int ch = from >> 7; ch <= (to >> 7); ch += 2) {
        const Win w = load_win(occ, row, ch);
        const int c = first_occupied(w, max(from, w.base), min(to, w.base + 255));
        if (c >= 0) return c;
    }
    return -1;
}
__device__ __forceinline__ int scan_behind(const uint4* occ, uint32_t row, int from, int to) {
    if (from > to) return -1;
    for (int ch = to >> 7; ch >= (from >> 7); ch -= 2) {
        const Win w = load_win(occ, row, max(ch - 1, 0));
        const int c = last_occupied(w, max(from, w.base), min(to, w.base + 255));
        if (c >= 0) return c;
    }
    return -1;
}
__device__ __forceinline__ uint32_t code_at(const uint8_t* codes, uint32_t row, int cell) {
    return __ldcg(codes + ((size_t)row << 7) + cell);
}

// Atlas cell address: the atlas holds < 2^32 cells (checked at ts_create), so (row, cell) packs
// into one 32-bit global cell index gc = row * 128 + cell.
__device__ __forceinline__ void atlas_vacate(const Ctx& c, uint32_t gc) {
    atomicAnd(reinterpret_cast<uint32_t*>(c.occ) + (gc >> 5), ~(1u << (gc & 31)));
}
// The bit that is already set when a cell is occupied is the by-product that proves invariant
// I2 (no two vehicles in one lane cell) on the device.
__device__ __forceinline__ void atlas_occupy(const Ctx& c, uint32_t gc, uint32_t code) {
    const uint32_t bit = 1u << (gc & 31);
    const uint32_t old = atomicOr(reinterpret_cast<uint32_t*>(c.occ) + (gc >> 5), bit);
    if (old & bit) atomicOr(&c.dyn->error, ERR_CELL_CLASH);
    c.codes[gc] = (uint8_t)code;
}

__device__ __forceinline__ unsigned long long mix64(unsigned long long z) {
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

__device__ __forceinline__ uint4 ldcg4(const uint4* p) { return __ldcg(p); }
__device__ __forceinline__ void stcg4(uint4* p, uint4 v) { __stcg(p, v); }

}  // namespace ts
