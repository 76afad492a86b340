// ts_device.cuh -- device-side data layout and the per-step phases of the traffic
// microsimulation (sections 6.3.2-6.3.3; rule set in DESIGN.md section 2).
//
// Product code for sm_100a.  Shares nothing with oracle/.  Built with -fmad=false and IEEE
// division so that every fp32 expression below is the written sequence of single operations.
//
// One simulation step k -> k+1 is two grid-wide phases:
//   phase_intent : every ACTIVE vehicle reads state k and the traffic atlas M_k (byte scans,
//                  16-byte vector loads), decides lane change / acceleration / crossing and
//                  posts step-tagged atomicMin claims; ready departure-queue heads do the same.
//   -- grid-wide dependency: all claims visible --
//   phase_commit : claims are resolved (lowest id wins), state k+1 is written, the vehicle's old
//                  atlas byte is erased and its new one stored (single buffer; race-free by
//                  invariant I6), arrivals retire, departures are appended, samples are taken.
//   -- grid-wide dependency: M_{k+1} complete --
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ts {

constexpr uint32_t NONE32 = 0xFFFFFFFFu;
enum : uint32_t { CTRL_FREE = 0, CTRL_PRIORITY = 1, CTRL_SIGNAL = 2 };
enum : uint32_t { ACT_STAY = 0, ACT_ARRIVE = 1, ACT_CROSS = 2 };
enum : uint32_t { ERR_CELL_CLASH = 1, ERR_SLOTS = 2 };

// 32 bytes per edge: everything a vehicle needs to know about the edge it is on (or enters),
// including the signal plan of the node at its head, in two 16-byte loads.
struct __align__(16) EdgeRec {
    uint32_t row16;      // atlas offset of lane 0's row, in 16-byte units
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

// Counters that change every step; one cache line in device memory.
struct Dyn {
    uint32_t n_pending, n_active, n_arrived;
    uint32_t slot_alloc;   // slots handed out so far (departures append here)
    uint32_t n_slots;      // slots visible to the step in flight
    uint32_t error;        // sticky ERR_*
    uint32_t n_samples;
    uint32_t k;            // step counter
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

// Everything the kernels touch.  Passed by value.
struct Ctx {
    Params p;
    uint32_t V, E, N, n_queues, cap_slots;
    // static network / demand
    const EdgeRec* edges;               // [E]
    const uint32_t* route_edges;        // [R]
    const uint32_t* route_begin;        // [V] first position of vehicle's route
    const uint32_t* route_end;          // [V] one past the last
    const float* v0_mult;               // [V]
    const float* mand_dist;             // [V]
    const uint32_t* queue_edge;         // [Q] origin edge of queue q
    const uint32_t* queue_off;          // [Q+1] into queue_veh / queue_dep
    const uint32_t* queue_veh;          // [V] ids ordered by (edge, dep_step, id)
    const uint32_t* queue_dep;          // [V] dep_step in the same order
    // mutable
    uint8_t* atlas;                     // traffic atlas, one byte per metre of lane
    uint32_t* queue_head;               // [Q]
    uint32_t* queue_cand;               // [Q] candidate id of this step or NONE32
    unsigned long long* lane_claim;     // [n_lanes] step-tagged minimum id
    unsigned long long* node_claim;     // [N]
    Dyn* dyn;
    // slot-ordered SoA of vehicles that have departed
    float* s_x; float* s_v; uint32_t* s_edge; uint32_t* s_meta;   // meta: lane | alive << 8
    uint32_t* s_id; uint32_t* s_next; uint32_t* s_rpos; uint32_t* s_enter;
    float* s_v0m; float* s_mand;
    float* s_xt; float* s_vt; uint32_t* s_act;                     // intent: act | lane_new << 4
    // id-ordered results
    uint8_t* o_status; uint8_t* o_lane; uint32_t* o_edge; float* o_x; float* o_v;
    uint32_t* o_rpos; uint32_t* o_insert; uint32_t* o_arrive;
    // per-edge statistics
    uint32_t* st_entered; uint32_t* st_exited; unsigned long long* st_exit_steps;
    uint32_t* st_samp_cnt; unsigned long long* st_samp_code;
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
__device__ __forceinline__ float idm_free(const Params& p, float v, float v0) {
    float r = v / v0;
    float r2 = r * r;
    float r4 = r2 * r2;
    return 1.0f - r4;
}
__device__ __forceinline__ float idm(const Params& p, float v, float v0, bool has, float s, float dv) {
    float fr = idm_free(p, v, v0);
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
__device__ __forceinline__ uint32_t stride16(const EdgeRec& e) { return ((uint32_t)e.len + 15u) >> 4; }
__device__ __forceinline__ const uint8_t* lane_row(const uint8_t* atlas, const EdgeRec& e, uint32_t lane) {
    return atlas + (((size_t)e.row16 + (size_t)lane * stride16(e)) << 4);
}

__device__ __forceinline__ unsigned long long claim_word(uint32_t k, uint32_t id) {
    // newer steps compare smaller, so a stale word never beats a live claim and nothing is cleared
    return ((unsigned long long)(0xFFFFFFFFu - k) << 32) | id;
}

// 16-bit mask of the non-zero bytes of a 16-byte chunk.
__device__ __forceinline__ uint32_t nz_mask(const uint4& q) {
    auto m4 = [](uint32_t w) -> uint32_t {
        uint32_t t = __vcmpne4(w, 0u);               // 0xFF per non-zero byte
        return (t & 1u) | ((t >> 7) & 2u) | ((t >> 14) & 4u) | ((t >> 21) & 8u);
    };
    return m4(q.x) | (m4(q.y) << 4) | (m4(q.z) << 8) | (m4(q.w) << 12);
}
__device__ __forceinline__ uint32_t chunk_byte(const uint4& q, int b) {
    uint32_t w = (b & 8) ? ((b & 4) ? q.w : q.z) : ((b & 4) ? q.y : q.x);
    return (w >> ((b & 3) * 8)) & 0xFFu;
}

// "we check the following bytes in memory": first occupied cell in [from, to]
// of a lane row, 16 bytes at a time.  Rows are 16-byte aligned and zero-padded to a multiple
// of 16, so an aligned chunk never leaves the row.  Returns the cell or -1.
__device__ __forceinline__ int scan_ahead(const uint8_t* row, int from, int to, uint32_t& code) {
    if (from > to) return -1;
    const uint4* r = reinterpret_cast<const uint4*>(row);
    for (int ch = from >> 4, last = to >> 4; ch <= last; ++ch) {
        uint4 q = __ldcg(r + ch);
        uint32_t m = nz_mask(q);
        int base = ch << 4;
        if (base < from) m &= 0xFFFFu << (from - base);
        if (base + 15 > to) m &= 0xFFFFu >> (base + 15 - to);
        if (m) { int b = __ffs((int)m) - 1; code = chunk_byte(q, b); return base + b; }
    }
    return -1;
}
// Last occupied cell in [from, to] (the lag vehicle), scanning backwards.
__device__ __forceinline__ int scan_behind(const uint8_t* row, int from, int to, uint32_t& code) {
    if (from > to) return -1;
    const uint4* r = reinterpret_cast<const uint4*>(row);
    for (int ch = to >> 4, first = from >> 4; ch >= first; --ch) {
        uint4 q = __ldcg(r + ch);
        uint32_t m = nz_mask(q);
        int base = ch << 4;
        if (base < from) m &= 0xFFFFu << (from - base);
        if (base + 15 > to) m &= 0xFFFFu >> (base + 15 - to);
        if (m) { int b = 31 - __clz((int)m); code = chunk_byte(q, b); return base + b; }
    }
    return -1;
}

__device__ __forceinline__ unsigned long long mix64(unsigned long long z) {
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

}  // namespace ts
