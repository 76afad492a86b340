// ts_phases.cuh -- the two phases of one simulation step as __device__ functions, so that the
// same code runs from the per-phase kernels and from the persistent cooperative kernel.
// Rule set and notation: DESIGN.md section 2 (steps 2a-2f, 3, 4, 5); citations per block.
//
// The step is latency-bound, so each function is written as a short chain
// of "trips" to L2: every load of a trip is issued before any of them is consumed.
//   intent : slot state -> edge records + own-lane window -> next-edge / target-lane windows
//            -> speed codes -> claims (fire and forget)
//   commit : slot state + intent -> [crossers only: edge records -> claims] -> stores
#pragma once
#include "ts_device.cuh"

namespace ts {

// ------------------------------------------------------------------ phase 1: intent

// DESIGN.md 2, step 2: one ACTIVE vehicle, reads state k and atlas M_k only.
__device__ __forceinline__ void vehicle_intent(const Ctx& c, uint32_t slot, uint32_t k) {
    const Params& p = c.p;
    // trip 1: slot state
    const uint32_t meta = __ldcg(c.s_meta + slot);
    if (!(meta >> 8)) return;
    const uint32_t l = meta & 0xFFu;
    const float x = __ldcg(c.s_x + slot), v = __ldcg(c.s_v + slot);
    const uint32_t e = __ldcg(c.s_edge + slot), e2 = __ldcg(c.s_next + slot);
    const uint32_t id = __ldcg(c.s_id + slot);
    const float v0m = __ldcg(c.s_v0m + slot);
    const uint32_t row = __ldcg(c.s_row + slot);
    const float mand = __ldcg(c.s_mand + slot);
    const int ci = (int)floorf(x);
    const bool fast = p.H <= 128 && p.Hb <= 128;      // one 256-cell window covers a scan

    // trip 2: edge records and the own-lane window
    const bool last = (e2 == NONE32);
    const EdgeRec E = load_edge(c.edges, e);
    EdgeRec E2 = E;
    if (!last) E2 = load_edge(c.edges, e2);
    Win w_own;
    if (fast) w_own = load_win(c.occ, row, (ci + 1) >> 7);

    // 2a
    const float v0 = v0m * E.vlim;
    const int C = E.len;
    const float Cf = (float)C;
    const uint32_t lanes = edge_lanes(E), lanes2 = edge_lanes(E2);
    const uint32_t l2 = l < lanes2 - 1 ? l : lanes2 - 1;
    const uint32_t ctrl = edge_ctrl(E);
    const bool may_cross = last || ctrl != CTRL_SIGNAL || signal_green(E, k);
    const int lim = min(C - 1, ci + p.H);
    const int Hp = p.H - (C - 1 - ci);
    const bool want_next = !last && may_cross && Hp > 0;
    const int lim2 = min((int)E2.len - 1, Hp - 1);
    const uint32_t row2 = lane_row(E2, l2);

    // 2d eligibility (readings R12, R14): known before any target-lane byte is read
    bool lc_eval = false;
    uint32_t lt = l, rowt = row;
    if (p.lc_period != 0 && lanes >= 2) {
        const int lti = (int)l + ((k & 1u) ? -1 : +1);
        float n = v + p.a_dt;
        n = n * p.dt;
        n = x + n;
        if (lti >= 0 && lti < (int)lanes && x >= p.entry_zone_f && n < Cf &&
            ((k >> 1) + id) % p.lc_period == 0) {
            lc_eval = true;
            lt = (uint32_t)lti;
            rowt = lane_row(E, lt);
        }
    }
    const int lo = max(0, ci - p.Hb);

    // trip 3: next-edge window and target-lane windows, all in flight together
    int cL = -1, cL2 = -1, cLt = -1, cF = -1;
    if (fast) {
        Win w_next, w_ta, w_tb;
        if (want_next) w_next = load_win(c.occ, row2, 0);
        if (lc_eval) { w_ta = load_win(c.occ, rowt, ci >> 7); w_tb = load_win(c.occ, rowt, lo >> 7); }
        cL = first_occupied(w_own, ci + 1, lim);                       // 2b
        if (cL < 0 && want_next) cL2 = first_occupied(w_next, 0, lim2);
        if (lc_eval) { cLt = first_occupied(w_ta, ci, lim); cF = last_occupied(w_tb, lo, ci - 1); }
    } else {
        cL = scan_ahead(c.occ, row, ci + 1, lim);
        if (cL < 0 && want_next) cL2 = scan_ahead(c.occ, row2, 0, lim2);
        if (lc_eval) { cLt = scan_ahead(c.occ, rowt, ci, lim); cF = scan_behind(c.occ, rowt, lo, ci - 1); }
    }

    // trip 4: speed codes of the vehicles found
    uint32_t code_lead = 1, code_Lt = 1, code_F = 1;
    if (cL >= 0) code_lead = code_at(c.codes, row, cL);
    else if (cL2 >= 0) code_lead = code_at(c.codes, row2, cL2);
    if (cLt >= 0) code_Lt = code_at(c.codes, rowt, cLt);
    if (cF >= 0) code_F = code_at(c.codes, rowt, cF);

    // 2b gaps (E3)
    const bool lead_on_edge = cL >= 0, has_lead = cL >= 0 || cL2 >= 0;
    float s_lead = 0.0f;
    if (lead_on_edge) {
        s_lead = (float)cL - p.len;
        s_lead = s_lead - x;
    } else if (has_lead) {
        s_lead = Cf - x;
        s_lead = s_lead + (float)cL2;
        s_lead = s_lead - p.len;
    }
    const float dv_lead = v - speed_decode(code_lead);

    // 2d gap acceptance G1-G3, then the mandatory rule or the MOBIL incentive G4
    bool accepted = false;
    const bool has_Lt = cLt >= 0;
    float s_Lt = 0.0f, at_c = 0.0f;
    if (lc_eval) {
        const bool has_F = cF >= 0;
        const float vLt = speed_decode(code_Lt), vF = speed_decode(code_F);
        float s_lag = 0.0f;
        if (has_Lt) { s_Lt = (float)cLt - p.len; s_Lt = s_Lt - x; }
        if (has_F) { s_lag = x - p.len; s_lag = s_lag - (float)(cF + 1); }
        bool ok = !has_Lt || s_Lt >= p.s0;                                   // G1
        float aF_new = 0.0f;
        if (ok && has_F) {                                                   // G2 (E4)
            float m = (vF + 0.125f) + p.half_a_dt;
            m = m * p.dt;
            ok = s_lag >= p.s0 && s_lag >= m;
        }
        if (ok && has_F) {                                                   // G3
            aF_new = idm(p, vF, E.vlim, true, s_lag, vF - v);
            ok = aF_new >= -p.b_safe;
        }
        if (ok) {                                                            // G4
            const float rem = Cf - x;
            at_c = idm(p, v, v0, has_Lt, s_Lt, v - vLt);
            if (!last && l >= lanes2 && lt < l && rem <= mand) accepted = true;
            else if (!last && lt >= lanes2 && rem <= mand) accepted = false;
            else {
                const float a_c = idm(p, v, v0, lead_on_edge, s_lead, dv_lead);
                float inc = at_c - a_c;
                if (has_F) {
                    float sF = (float)cLt - p.len;
                    sF = sF - (float)(cF + 1);
                    const float a_F = idm(p, vF, E.vlim, has_Lt, sF, vF - vLt);
                    float d2 = aF_new - a_F;
                    d2 = p.politeness * d2;
                    inc = inc + d2;
                }
                accepted = inc > p.lc_threshold;
            }
        }
    }

    // 2e acceleration (min over leader, stop line, new-lane leader) and integration (E2)
    float acc = idm(p, v, v0, has_lead, s_lead, dv_lead);
    if (!may_cross) acc = fminf(acc, idm(p, v, v0, true, Cf - x, v));             // 2c
    float cap = __int_as_float(0x7f800000);
    if (has_lead) cap = fmaxf(s_lead, 0.0f);
    if (accepted && has_Lt) { acc = fminf(acc, at_c); cap = fminf(cap, fmaxf(s_Lt, 0.0f)); }
    float vt = acc * p.dt;
    vt = v + vt;
    vt = fmaxf(vt, 0.0f);
    vt = fminf(vt, v0);
    float dx = v + vt;
    dx = 0.5f * dx;
    dx = dx * p.dt;
    if (dx > cap) { dx = cap; vt = 0.0f; }
    float xt = x + dx;

    // 2f crossing intent and claims (one vehicle at a time; lowest id wins)
    uint32_t act = ACT_STAY, nrow = accepted ? rowt : row;
    if (xt >= Cf) {
        if (last) act = ACT_ARRIVE;
        else if (may_cross) {
            act = ACT_CROSS;
            nrow = row2;
            const unsigned long long w = claim_word(k, id);
            atomicMin(c.lane_claim + E2.lane_base + l2, w);
            if (ctrl == CTRL_PRIORITY) atomicMin(c.node_claim + E.to_node, w);
        } else { xt = Cf - 0.0625f; vt = 0.0f; }
    }
    c.s_xt[slot] = xt;
    c.s_vt[slot] = vt;
    c.s_act[slot] = act | ((accepted ? lt : l) << 4);
    c.s_nrow[slot] = nrow;
}

// DESIGN.md 2, step 3: the head of one departure queue.
__device__ __forceinline__ void departure_intent(const Ctx& c, uint32_t q, uint32_t k) {
    uint32_t cand = NONE32;
    const uint32_t head = __ldcg(c.queue_head + q);
    if (head < __ldg(c.queue_off + q + 1) && __ldg(c.queue_dep + head) <= k) {
        const EdgeRec E = load_edge(c.edges, __ldg(c.queue_edge + q));
        const Win w = load_win(c.occ, E.row, 0);
        if (first_occupied(w, 0, (int)c.p.insert_clear - 1) < 0) {
            cand = __ldg(c.queue_veh + head);
            atomicMin(c.lane_claim + E.lane_base, claim_word(k, cand));
        }
    }
    c.queue_cand[q] = cand;
}

__device__ __forceinline__ void phase_intent(const Ctx& c, uint32_t k, uint32_t tid, uint32_t nthreads) {
    const uint32_t n_slots = __ldcg(&c.dyn->slot_alloc);   // nothing appends during this phase
    if (tid == 0) {
        c.dyn->n_slots = n_slots;
        // every vehicle ACTIVE at step k is advanced once: the metric's unit of work
        c.dyn->updates += __ldcg(&c.dyn->n_active);
    }
    for (uint32_t s = tid; s < n_slots; s += nthreads) vehicle_intent(c, s, k);
    for (uint32_t q = tid; q < c.n_queues; q += nthreads) departure_intent(c, q, k);
}

// ------------------------------------------------------------------ phase 2: resolve + commit

// Vacate (row_from, cell_from) and occupy (row_to, cell_to) with `code`.  Single buffer: no other
// vehicle's new cell equals this vehicle's old cell (invariant I6), and bit updates commute, so
// the integer atomics of different threads never conflict.  The bit that is already set when a
// cell is occupied is the by-product that proves invariant I2 on the device.
__device__ __forceinline__ void atlas_move(const Ctx& c, bool has_from, uint32_t row_from, int cell_from,
                                           uint32_t row_to, int cell_to, uint32_t code) {
    uint32_t* occ32 = reinterpret_cast<uint32_t*>(c.occ);
    if (!has_from || row_from != row_to || cell_from != cell_to) {
        if (has_from) atomicAnd(occ32 + ((size_t)row_from << 2) + (cell_from >> 5), ~(1u << (cell_from & 31)));
        const uint32_t bit = 1u << (cell_to & 31);
        const uint32_t old = atomicOr(occ32 + ((size_t)row_to << 2) + (cell_to >> 5), bit);
        if (old & bit) atomicOr(&c.dyn->error, ERR_CELL_CLASH);
    }
    c.codes[((size_t)row_to << 7) + cell_to] = (uint8_t)code;
}

__device__ __forceinline__ void vehicle_commit(const Ctx& c, uint32_t slot, uint32_t k, bool sample) {
    // trip 1: slot state and intent
    const uint32_t meta = __ldcg(c.s_meta + slot);
    if (!(meta >> 8)) return;
    const uint32_t l = meta & 0xFFu;
    const uint32_t a = __ldcg(c.s_act + slot);
    const uint32_t e = __ldcg(c.s_edge + slot);
    const float x_old = __ldcg(c.s_x + slot);
    float xn = __ldcg(c.s_xt + slot), vn = __ldcg(c.s_vt + slot);
    const uint32_t row = __ldcg(c.s_row + slot);
    uint32_t nrow = __ldcg(c.s_nrow + slot);
    const uint32_t act = a & 15u;
    uint32_t l_new = a >> 4, e_new = e;
    const uint32_t k1 = k + 1;
    const int c_old = (int)floorf(x_old);

    if (act != ACT_STAY) {
        const uint32_t id = __ldcg(c.s_id + slot);
        const uint32_t e2 = __ldcg(c.s_next + slot);
        const uint32_t enter = __ldcg(c.s_enter + slot);
        const uint32_t rpos = __ldcg(c.s_rpos + slot);
        const EdgeRec E = load_edge(c.edges, e);
        if (act == ACT_CROSS) {
            // trip 2: edge records and the route two edges ahead; trip 3: the claim words
            const EdgeRec E2 = load_edge(c.edges, e2);
            const uint32_t rend = __ldg(c.route_end + id);
            const uint32_t e3 = (rpos + 2 < rend) ? __ldg(c.route_edges + rpos + 2) : NONE32;
            const float v0m = __ldcg(c.s_v0m + slot);
            const uint32_t lanes2 = edge_lanes(E2);
            const uint32_t l2 = l < lanes2 - 1 ? l : lanes2 - 1;
            const unsigned long long w = claim_word(k, id);
            const unsigned long long wl = __ldcg(c.lane_claim + E2.lane_base + l2);
            const unsigned long long wn = (edge_ctrl(E) == CTRL_PRIORITY) ? __ldcg(c.node_claim + E.to_node) : w;
            const float Cf = (float)E.len;
            if (wl == w && wn == w) {                  // holds every claim it made: crosses
                xn = xn - Cf;
                xn = fminf(xn, (float)E2.len - 0.0625f);
                vn = fminf(vn, v0m * E2.vlim);         // R9
                e_new = e2; l_new = l2;
                c.s_rpos[slot] = rpos + 1;
                c.s_next[slot] = e3;
                c.s_edge[slot] = e2;
                c.s_enter[slot] = k1;
                atomicAdd(c.st_entered + e2, 1u);
                atomicAdd(c.st_exited + e, 1u);
                atomicAdd(c.st_exit_steps + e, (unsigned long long)(k1 - enter));
            } else {                                   // lost a claim: held at the line (R15)
                xn = Cf - 0.0625f; vn = 0.0f; l_new = l; nrow = row;
            }
        } else {                                       // ACT_ARRIVE
            atomicAnd(reinterpret_cast<uint32_t*>(c.occ) + ((size_t)row << 2) + (c_old >> 5), ~(1u << (c_old & 31)));
            c.s_meta[slot] = l;                        // alive bit off
            c.o_status[id] = 2; c.o_arrive[id] = k1; c.o_x[id] = (float)E.len; c.o_v[id] = vn;
            c.o_edge[id] = e; c.o_lane[id] = (uint8_t)l; c.o_rpos[id] = rpos;
            atomicAdd(c.st_exited + e, 1u);
            atomicAdd(c.st_exit_steps + e, (unsigned long long)(k1 - enter));
            atomicSub(&c.dyn->n_active, 1u);
            atomicAdd(&c.dyn->n_arrived, 1u);
            atomicAdd(&c.dyn->sum_arrive, (unsigned long long)k1);
            return;
        }
    }
    c.s_x[slot] = xn;
    c.s_v[slot] = vn;
    if (l_new != l) c.s_meta[slot] = l_new | 0x100u;
    if (nrow != row) c.s_row[slot] = nrow;
    const uint32_t code = speed_code(vn);
    atlas_move(c, true, row, c_old, nrow, (int)floorf(xn), code);
    if (sample) {                                      // PAPER.md:437 one sample per minute
        atomicAdd(c.st_samp_cnt + e_new, 1u);
        atomicAdd(c.st_samp_code + e_new, (unsigned long long)(code - 1));
    }
}

// DESIGN.md 2, step 4 (departures): the winning queue head becomes ACTIVE at x = 0, v = 0, lane 0.
__device__ __forceinline__ void departure_commit(const Ctx& c, uint32_t q, uint32_t k, bool sample) {
    const uint32_t id = __ldcg(c.queue_cand + q);
    if (id == NONE32) return;
    const uint32_t e = __ldg(c.queue_edge + q);
    const EdgeRec E = load_edge(c.edges, e);
    if (__ldcg(c.lane_claim + E.lane_base) != claim_word(k, id)) return;
    const uint32_t slot = atomicAdd(&c.dyn->slot_alloc, 1u);
    if (slot >= c.cap_slots) { atomicOr(&c.dyn->error, ERR_SLOTS); return; }
    const uint32_t k1 = k + 1;
    const uint32_t rb = __ldg(c.route_begin + id);
    c.s_x[slot] = 0.0f; c.s_v[slot] = 0.0f; c.s_edge[slot] = e; c.s_meta[slot] = 0x100u;
    c.s_id[slot] = id; c.s_rpos[slot] = rb; c.s_enter[slot] = k1; c.s_row[slot] = E.row;
    c.s_next[slot] = (rb + 1 < __ldg(c.route_end + id)) ? __ldg(c.route_edges + rb + 1) : NONE32;
    c.s_v0m[slot] = __ldg(c.v0_mult + id); c.s_mand[slot] = __ldg(c.mand_dist + id);
    c.o_status[id] = 1; c.o_insert[id] = k1;
    c.queue_head[q] = __ldcg(c.queue_head + q) + 1;
    atlas_move(c, false, 0, 0, E.row, 0, 1u);
    atomicAdd(c.st_entered + e, 1u);
    atomicSub(&c.dyn->n_pending, 1u);
    atomicAdd(&c.dyn->n_active, 1u);
    if (sample) atomicAdd(c.st_samp_cnt + e, 1u);  // speed code - 1 == 0 at rest
}

__device__ __forceinline__ void phase_commit(const Ctx& c, uint32_t k, uint32_t tid, uint32_t nthreads) {
    const uint32_t n_slots = __ldcg(&c.dyn->n_slots);
    const bool sample = c.p.sample_period && ((k + 1) % c.p.sample_period == 0);
    if (tid == 0) { c.dyn->k = k + 1; if (sample) c.dyn->n_samples += 1; }
    for (uint32_t s = tid; s < n_slots; s += nthreads) vehicle_commit(c, s, k, sample);
    for (uint32_t q = tid; q < c.n_queues; q += nthreads) departure_commit(c, q, k, sample);
}

}  // namespace ts
