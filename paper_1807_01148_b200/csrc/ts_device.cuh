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
//   code plane : the occupant's speed code (valid only where occupied), one byte per GRANULE of
//                2^cg cells: 4 cells where vehicles are at least 4 m long (two vehicles of a lane are
//                then never in one granule, see Params::cg), else one byte per cell;
//   occupancy  : one bit per cell, 16 bytes per chunk, so that "check the following bytes" for a
//                128-cell lookahead is two independent 16-byte loads and an __ffs instead of a
//                chain of up to nine dependent loads.
// Vacating a cell clears its bit only; stale code bytes are never read.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ts {

constexpr uint32_t NONE32 = 0xFFFFFFFFu;
// CTRL_STOP: stop control with a persistent node owner (reading R34); CTRL_SIGNAL_NM:
// one signal phase per movement (inbound edge, outbound edge) ("combination nm"; R35)
enum : uint32_t { CTRL_FREE = 0, CTRL_PRIORITY = 1, CTRL_SIGNAL = 2, CTRL_STOP = 3, CTRL_SIGNAL_NM = 4 };
enum : uint32_t { ERR_CELL_CLASH = 1, ERR_SLOTS = 2, ERR_LOGIC = 4, ERR_NAN = 8, ERR_SPACING = 16 };
// flags in Slots::A.w above the lane number: the vehicle takes part in the steps; has made its stop
// at the STOP line of its edge; holds the STOP node at the tail of its edge; its type
enum : uint32_t { ALIVE = 0x100u, STOPPED = 0x200u, OWNS = 0x400u, TYPE_SHIFT = 12, TYPE_MASK = 0x3000u };
constexpr int kMaxTypes = 4;
// move-record kinds (uint4.w)
enum : uint32_t { MR_NONE = 0, MR_MOVE = 1, MR_CLEAR = 2, MR_CROSS = 3 };

// 32 bytes per edge: everything a vehicle needs to know about the edge it is on (or enters),
// including the signal plan of the node at its head, in two 16-byte loads.
struct __align__(32) EdgeRec {
    uint32_t row;        // atlas offset of lane 0's row, in chunks of 128 cells
    uint32_t lane_base;  // global lane index of lane 0 (index of its claim word)
    float vlim;          // m/s
    uint32_t to_node;
    // Signal plan of the head node, reduced on the host to "green iff (k + off) mod cycle < green"
    // (off = offset - in_rank * (green + allred), mod cycle), with the modulo by the run-time
    // invariant `cycle` done by multiplication (Granlund & Montgomery 1994, N = 32):
    //   t = mulhi(magic, n);  q = (t + ((n - t) >> sh1)) >> sh2;  n mod cycle = n - q * cycle.
    uint32_t cyc_lc;     // cycle (n_in * (green + allred), < 2^24; 1 where not SIGNAL) | lanes << 24 | ctrl << 28
    uint32_t off_sh;     // off (< cycle) | sh1 << 24 | sh2 << 25
    uint32_t magic;      // floor(2^32 (2^l - cycle) / cycle) + 1, l = ceil(log2 cycle)
    uint16_t green;      // steps
    uint16_t len;        // cells
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
    // option "profile": nanoseconds CTA 0 spent in { phase 1, barrier 1, phase 2, barrier 2,
    // compaction + re-sort, digest }, and the number of steps they cover
    unsigned long long prof[8];
    // adaptive CTA size: which of the two instantiations enqueued for a chunk of steps should run
    // (0 = the spill-free small one, 1 = the one with more warps).  Chunk c reads word c & 1 and
    // writes the other one, so the second launch of a chunk never sees the first one's verdict on
    // the NEXT chunk; see run_steps()
    uint32_t prefer_big[2];
};

struct Params {
    float dt, a, b, T, s0, len, b_safe, politeness, lc_threshold;
    float Kinv;            // 1 / (2*sqrtf(a*b)), computed once on the host in fp32 (reading R27)
    float half_a_dt;       // (0.5f*a)*dt   (E4)
    float a_dt;            // a*dt          (E5)
    float entry_zone_f;
    int H, Hb;
    uint32_t lc_period, insert_clear, sample_period;
    uint32_t lc_pow2;      // lc_period is a power of two: the stagger test is a mask
    float inv_dt;          // 1 / dt, rounded once on the host (reading R30)
    // extended rule set (template parameter EXT of the phases): vehicle types (R31) ...
    float t_len[kMaxTypes], t_a[kMaxTypes], t_Kinv[kMaxTypes], t_a_dt[kMaxTypes], t_half_a_dt[kMaxTypes], t_vmax[kMaxTypes];
    // ... and control variants (R34-R36)
    float two_b;           // 2*b (amber: go on iff v^2 > 2 b (C - x))
    float stop_dist, stop_speed;
    uint32_t amber;        // steps of amber after every green
    // code plane (and type plane): one byte per 2^cg cells of a lane row.  cg = 2 where no two vehicles of a
    // lane can sit within 4 cells of each other (every vehicle at least 4 m long, insert_clear >= 4: see
    // code_granule_shift() in ts_api.cu), else 0.
    uint32_t cg;
};
// a sample is taken with the state after every sample_period-th step.
__device__ __forceinline__ bool sample_step(const Params& p, uint32_t k) {
    return p.sample_period && ((k + 1) % p.sample_period == 0);
}

// Slot-ordered vehicle state: three 16-byte vectors per slot (two ping-pong sets, swapped by
// the re-sort).
//   A = { bits(x), bits(v), row (first chunk of the vehicle's lane row), lane | ALIVE }
//   B = { edge, next route edge or NONE32, vehicle id, bits(v0_mult) }
//   C = { route position, one past the last route position, step it entered the edge, bits(mand_dist) }
//   D = { grams of CO, millilitres of fuel } so far (section 6.3.4; nullptr when not kept)
struct Slots {
    uint4* A;
    uint4* B;
    uint4* C;
    float2* D;
};

// Everything the kernels touch.  Passed by value.
struct Ctx {
    Params p;
    uint32_t V, E, N, n_queues, cap_slots;
    uint32_t sort_groups;               // re-sort key = (id & (sort_groups - 1)) * E + edge
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
    uint32_t* hist;                     // [sort_groups * E]
    uint32_t* base;                     // [sort_groups * E]
    unsigned long long* audit;          // [2] occupied cells counted / vehicles whose cell is not marked
    uint32_t* partial;                  // [kMaxCtas]
    // id-ordered results
    uint8_t* o_status; uint8_t* o_lane; uint32_t* o_edge; float* o_x; float* o_v;
    uint32_t* o_rpos; uint32_t* o_insert; uint32_t* o_arrive;
    // per-edge statistics
    uint32_t* st_entered; uint32_t* st_exited; unsigned long long* st_exit_steps;
    uint32_t* st_samp_cnt; unsigned long long* st_samp_code;
    // section 6.3.4 totals, id-ordered { grams of CO, millilitres of fuel }: written when a vehicle
    // arrives and by ts_read_emissions' gather (while it drives they live in Slots::D); nullptr = not kept
    float2* emis;
    // extended rule set only (nullptr otherwise)
    uint8_t* types;                     // traffic atlas, type plane: the occupant's vehicle type (valid where occupied)
    const uint32_t* edge_aux;           // [E] phase length P of the head node's signal | rank among the tail node's outbound edges << 16
    const uint32_t* edge_from;          // [E] tail node
    uint32_t* node_free_from;           // [N] CTRL_STOP: first step at which the node is free again (UINT32_MAX while held)
};

constexpr uint32_t kMaxCtas = 2048;

// Who am I in the grid: slots are dealt to CTAs in tiles of blockDim.x consecutive slots, round
// robin, so that consecutive (edge-sorted) slots sit in consecutive lanes of one warp.
struct Who {
    uint32_t t, T, cta, n_cta;
    // Slots (and departure queues) are dealt out in tiles of 32 -- one warp -- round robin over the
    // CTAs first and the warps of a CTA second: a few thousand vehicles spread over all SMs (the
    // step is bound by latency then), and consecutive edge-sorted slots share a warp.
    __device__ __forceinline__ uint32_t slot(uint32_t j) const {
        return ((j * (T >> 5) + (t >> 5)) * n_cta + cta) * 32u + (t & 31u);
    }
    // Departure queues are dealt the same way but to the warps of a CTA in REVERSE order: the first
    // warps are the ones that get one more tile of vehicles whenever the tiles do not divide evenly,
    // so the queue heads (an L2 round trip of their own in each phase) go to the warps with slack.
    __device__ __forceinline__ uint32_t qslot(uint32_t j) const {
        const uint32_t W = T >> 5;
        return ((j * W + (W - 1u - (t >> 5))) * n_cta + cta) * 32u + (t & 31u);
    }
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
    float rinv = __frcp_rn(v0);                     // the correctly rounded 1.0f / v0 (reading R27)
    float r = v * rinv;
    float r2 = r * r;
    float r4 = r2 * r2;
    return 1.0f - r4;
}
// `a`, `Kinv`: the subject vehicle's acceleration ability and 1 / (2 sqrt(a b)) (per type).
__device__ __forceinline__ float idm(const Params& p, float a, float Kinv, float v, float v0, bool has, float s, float dv) {
    float fr = idm_free(v, v0);
    if (!has) return a * fr;
    float t = v * p.T;
    float u = v * dv;
    float w = u * Kinv;
    t = t + w;
    t = fmaxf(t, 0.0f);
    float ss = p.s0 + t;
    float se = fmaxf(s, 0.5f);
    float q = ss / se;
    float q2 = q * q;
    float d = fr - q2;
    return a * d;
}
// The same in two pieces, so that the free-road factor of one (v, v0) is formed once and several
// interactions are evaluated side by side (independent chains: the scheduler overlaps them).
__device__ __forceinline__ float idm_follow(const Params& p, float a, float Kinv, float fr, float v, float s, float dv) {
    float t = v * p.T;
    float u = v * dv;
    float w = u * Kinv;
    t = t + w;
    t = fmaxf(t, 0.0f);
    float ss = p.s0 + t;
    float se = fmaxf(s, 0.5f);
    float q = ss / se;
    float q2 = q * q;
    float d = fr - q2;
    return a * d;
}

// Section 6.3.4.  Eq. 8: grams of CO per second at speed v; the paper's v_m is
// in miles per hour, 1 m/s = 2.2369363 mph (reading R28).
__device__ __forceinline__ float co_rate(float v) {
    const float vm = v * 2.2369363f;
    const float off = vm - 50.0f;
    const float lin = -0.064f + 0.0056f * vm;
    return lin + 0.00026f * (off * off);
}
// Eq. 9: millilitres of fuel per second at speed v (m/s) and acceleration acc (m/s^2); the engine
// drag term only while accelerating, the power demand floored at zero (reading R29).
__device__ __forceinline__ float fuel_rate(float v, float acc) {
    const float v2 = v * v;
    float dem = 0.269f * v + 0.0171f * v2;
    dem = dem + 0.000672f * (v2 * v);
    dem = dem + (1.680f * acc) * v;
    if (acc > 0.0f) dem = dem + (0.79296f * (acc * acc)) * v;
    dem = fmaxf(dem, 0.0f);
    return 0.666f + 0.072f * dem;
}

// Steps since this inbound edge's (or, with `shift`, this movement's) phase began, modulo the cycle:
// green while < green, then amber for Params::amber steps, then red.  `shift` < cycle.
__device__ __forceinline__ uint32_t signal_pos(const EdgeRec& e, uint32_t k, uint32_t shift = 0u) {
    const uint32_t cycle = e.cyc_lc & 0xFFFFFFu;
    const uint32_t n = k + (e.off_sh & 0xFFFFFFu) + shift;   // k < 2^31, off, shift < 2^24
    const uint32_t t = __umulhi(e.magic, n);
    const uint32_t q = (t + ((n - t) >> ((e.off_sh >> 24) & 1u))) >> (e.off_sh >> 25);
    return n - q * cycle;
}
__device__ __forceinline__ bool signal_green(const EdgeRec& e, uint32_t k) {
    return signal_pos(e, k) < (uint32_t)e.green;
}

// One 256-bit load (sm_100 LDG.256): a record is one 32-byte sector, and a warp whose vehicles sit
// on 20 different edges pays for 20 sectors once instead of twice.
__device__ __forceinline__ EdgeRec load_edge(const EdgeRec* edges, uint32_t e) {
    EdgeRec r;
    uint32_t* w = reinterpret_cast<uint32_t*>(&r);
    asm("ld.global.nc.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
        : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]), "=r"(w[4]), "=r"(w[5]), "=r"(w[6]), "=r"(w[7])
        : "l"(edges + e));
    return r;
}
__device__ __forceinline__ uint32_t edge_lanes(const EdgeRec& e) { return (e.cyc_lc >> 24) & 15u; }
__device__ __forceinline__ uint32_t edge_ctrl(const EdgeRec& e) { return e.cyc_lc >> 28; }
__device__ __forceinline__ uint32_t row_stride(const EdgeRec& e) { return ((uint32_t)e.len + 127u) >> 7; }
__device__ __forceinline__ uint32_t lane_row(const EdgeRec& e, uint32_t lane) { return e.row + lane * row_stride(e); }

__device__ __forceinline__ unsigned long long claim_word(uint32_t k, uint32_t id) {
    // newer steps compare smaller, so a stale word never beats a live claim and nothing is cleared
    return ((unsigned long long)(0xFFFFFFFFu - k) << 32) | id;
}

// ---- occupancy windows: 256 cells = two 16-byte chunks of one lane row, loaded together ----
struct Win {
    uint4 a, b;   // chunk ch and chunk ch+1
};
// `row` = first chunk of the lane row, `ch` = first chunk wanted (-1 is legal: the plane has one
// spare chunk in front and two behind).  Both loads are unconditional: a neighbouring chunk may
// belong to another lane's row; callers bound the RESULT by the cells they may look at, so no
// clamping -- and no dependence on the edge record -- is needed before the loads are issued.
__device__ __forceinline__ Win load_win(const uint4* occ, uint32_t row, int ch) {
    Win w;
    const uint4* p = occ + (ptrdiff_t)row + ch;
    w.a = __ldcg(p);
    w.b = __ldcg(p + 1);
    return w;
}
// 160 bits of the window starting at bit f (0 <= f < 128): a[0] bit 0 is window bit f.  A two-
// stage word barrel plus funnel shifts: no dynamic register indexing, no per-word masks.
struct Bits160 { uint32_t a0, a1, a2, a3, a4; };
__device__ __forceinline__ Bits160 extract160(const Win& w, int f) {
    uint32_t w0 = w.a.x, w1 = w.a.y, w2 = w.a.z, w3 = w.a.w, w4 = w.b.x, w5 = w.b.y, w6 = w.b.z, w7 = w.b.w;
    if (f & 64) { w0 = w2; w1 = w3; w2 = w4; w3 = w5; w4 = w6; w5 = w7; }
    if (f & 32) { w0 = w1; w1 = w2; w2 = w3; w3 = w4; w4 = w5; }
    const uint32_t sh = (uint32_t)f & 31u;
    Bits160 r;
    r.a0 = __funnelshift_r(w0, w1, sh);
    r.a1 = __funnelshift_r(w1, w2, sh);
    r.a2 = __funnelshift_r(w2, w3, sh);
    r.a3 = __funnelshift_r(w3, w4, sh);
    r.a4 = w4 >> sh;
    return r;
}
// "we check the following bytes in memory": the first occupied cell among the n
// cells (n <= 129) that start at cell `from`; `w` must hold the chunk of `from` and the one after.
// Returns the cell index or -1.  Bits beyond the n-th need no masking: if the first set bit lies
// beyond them, none lies within.
__device__ __forceinline__ int first_occupied(const Win& w, int from, int n) {
    const Bits160 b = extract160(w, from & 127);
    // branch-free: pick the first non-zero word, then one find-first-set
    uint32_t word = b.a4 & 1u;
    int base = 128;
    if (b.a3) { word = b.a3; base = 96; }
    if (b.a2) { word = b.a2; base = 64; }
    if (b.a1) { word = b.a1; base = 32; }
    if (b.a0) { word = b.a0; base = 0; }
    const int pos = word ? base + __ffs((int)word) - 1 : 192;
    return pos < n ? from + pos : -1;
}
// The last occupied cell among the n cells (n <= 128) that END at cell `last` (the lag vehicle,
// PAPER.md:400); `w` must hold the chunk before the chunk of `last`, and the chunk of `last`.
__device__ __forceinline__ int last_occupied(const Win& w, int last, int n) {
    // window bit of `last` is 128 + (last & 127); take the 160 bits that start 128 below it, so
    // that `last` is bit 128 of them and the cell d behind it is bit 128 - d
    const Bits160 b = extract160(w, last & 127);
    uint32_t word = b.a0 & ~1u;                        // bit 0 would be 128 cells behind: out of range
    int top = 31;                                      // bit index (of the 160) of the word's bit 31
    if (b.a1) { word = b.a1; top = 63; }
    if (b.a2) { word = b.a2; top = 95; }
    if (b.a3) { word = b.a3; top = 127; }
    int back = word ? 128 - (top - __clz((int)word)) : 192;
    if (b.a4 & 1u) back = 0;
    return back < n ? last - back : -1;
}
// General ranges (lookahead > 128 cells): 128 cells at a time.
__device__ __forceinline__ int scan_ahead(const uint4* occ, uint32_t row, int from, int to) {
    for (; from <= to; from += 128) {
        const int c = first_occupied(load_win(occ, row, from >> 7), from, min(128, to - from + 1));
        if (c >= 0) return c;
    }
    return -1;
}
__device__ __forceinline__ int scan_behind(const uint4* occ, uint32_t row, int from, int to) {
    for (; to >= from; to -= 128) {
        const int c = last_occupied(load_win(occ, row, (to >> 7) - 1), to, min(128, to - from + 1));
        if (c >= 0) return c;
    }
    return -1;
}
__device__ __forceinline__ uint32_t code_at(const uint8_t* codes, uint32_t row, int cell, uint32_t cg) {
    return __ldcg(codes + ((((size_t)row << 7) + cell) >> cg));
}

// Atlas cell address: the atlas holds < 2^32 cells (checked at ts_create), so (row, cell) packs
// into one 32-bit global cell index gc = row * 128 + cell.
//
// Moving a vehicle vacates its old cell and occupies its new one with fire-and-forget integer
// reductions (no return value is waited for).  Single buffer: no other vehicle's new cell equals
// this vehicle's old cell (invariant I6) and bit updates commute, so threads never conflict.
// Invariant I2 (no two vehicles in one lane cell) is audited when the state is read back
// (k_audit): every ACTIVE vehicle's cell is marked and the number of marked cells equals the
// number of ACTIVE vehicles.
__device__ __forceinline__ void atlas_move(const Ctx& c, uint32_t gc_from, uint32_t gc_to, uint32_t code) {
    uint32_t* occ32 = reinterpret_cast<uint32_t*>(c.occ);
    if (gc_from != gc_to) {
        const uint32_t bf = 1u << (gc_from & 31), bt = 1u << (gc_to & 31);
        if ((gc_from >> 5) == (gc_to >> 5)) atomicXor(occ32 + (gc_to >> 5), bf | bt);
        else { atomicAnd(occ32 + (gc_from >> 5), ~bf); atomicOr(occ32 + (gc_to >> 5), bt); }
    }
    c.codes[gc_to >> c.p.cg] = (uint8_t)code;
}
// extended rule set: the occupant's type travels with its speed code (`code_type` = code | type << 8)
__device__ __forceinline__ void atlas_set_type(const Ctx& c, uint32_t gc, uint32_t code_type) {
    if (c.types) c.types[gc >> c.p.cg] = (uint8_t)(code_type >> 8);
}
__device__ __forceinline__ uint32_t type_at(const uint8_t* types, uint32_t row, int cell, uint32_t cg) {
    return __ldcg(types + ((((size_t)row << 7) + cell) >> cg));
}
__device__ __forceinline__ void atlas_vacate(const Ctx& c, uint32_t gc) {
    atomicAnd(reinterpret_cast<uint32_t*>(c.occ) + (gc >> 5), ~(1u << (gc & 31)));
}
__device__ __forceinline__ void atlas_occupy(const Ctx& c, uint32_t gc, uint32_t code) {
    atomicOr(reinterpret_cast<uint32_t*>(c.occ) + (gc >> 5), 1u << (gc & 31));
    c.codes[gc >> c.p.cg] = (uint8_t)code;
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
