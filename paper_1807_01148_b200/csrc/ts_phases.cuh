// ts_phases.cuh -- the two phases of one simulation step as __device__ functions, so that the
// same code runs from the per-phase kernels and from the persistent cooperative kernel.
// Rule set and notation: DESIGN.md section 2 (steps 2a-2f, 3, 4, 5); citations per block.
//
// Each function is written as a short chain of "trips" to L2: every load of a trip is issued
// before any of them is consumed.
//   phase 1 : slot state (A, B) -> edge records + own-lane window [+ C if it may leave the edge or
//             evaluates a lane change] -> next-edge / target-lane windows [+ route entry] -> speed
//             codes -> own state k+1, move record, claims (fire and forget)
//   phase 2 : move record (shared memory) -> atlas update (fire and forget); crossing vehicles:
//             claim words + crossing record + state in ONE trip -> stores
#pragma once
#include "ts_device.cuh"

namespace ts {

// ------------------------------------------------------------------ phase 1: vehicles

// DESIGN.md 2, steps 2a-2f for one slot.  Reads state k and atlas M_k only; returns the move
// record that phase 2 applies.  `n_upd` counts ACTIVE vehicles advanced (the metric's unit).
// EMIS: keep the section 6.3.4 totals (compiled out of the default instantiation).
// EXT: the extended rule set -- vehicle types (reading R31: own length, acceleration
//      ability and speed cap; gaps use the length of the vehicle ahead, read from the atlas's type
//      plane) and the control variants of PAPER.md:402 (R34 STOP with a persistent node owner, R35 one
//      signal phase per movement, R36 amber).  Compiled out of the default instantiation, which is
//      instruction for instruction the code without them.
template <bool EMIS, bool EXT>
__device__ __forceinline__ uint4 vehicle_phase1(const Ctx& c, const Slots& S, uint32_t slot, uint32_t k,
                                                bool sample, uint32_t& n_upd) {
    const Params& p = c.p;
    // trip 1: slot state
    const uint4 sa = ldcg4(S.A + slot);
    const uint4 sb = ldcg4(S.B + slot);
    float2 em = make_float2(0.0f, 0.0f);               // section 6.3.4 totals so far (slot-ordered: coalesced)
    if (EMIS) em = __ldcg(S.D + slot);
    if (!(sa.w & ALIVE)) return make_uint4(0, 0, 0, MR_NONE);
    n_upd++;
    const float x = __uint_as_float(sa.x), v = __uint_as_float(sa.y);
    const uint32_t row = sa.z, l = sa.w & 0xFu;
    const uint32_t e = sb.x, e2 = sb.y, id = sb.z;
    const float v0m = __uint_as_float(sb.w);
    const int ci = (int)floorf(x);
    const bool fast = p.H <= 128 && p.Hb <= 128;      // one 256-cell window covers a scan
    // this vehicle's type (EXT) or the one type there is
    const uint32_t ty = EXT ? (sa.w & TYPE_MASK) >> TYPE_SHIFT : 0u;
    const float len_i = EXT ? p.t_len[ty] : p.len, a_i = EXT ? p.t_a[ty] : p.a, Kinv_i = EXT ? p.t_Kinv[ty] : p.Kinv;
    const float a_dt_i = EXT ? p.t_a_dt[ty] : p.a_dt;
    uint32_t flags = EXT ? (sa.w & (TYPE_MASK | STOPPED | OWNS)) : 0u;     // travels with the slot

    // trip 2: edge records and the own-lane window
    const bool last = (e2 == NONE32);
    const EdgeRec E = load_edge(c.edges, e);
    const EdgeRec E2 = load_edge(c.edges, last ? e : e2);      // no branch: the last edge stands in for itself
    Win w_own;
    if (fast) w_own = load_win(c.occ, row, (ci + 1) >> 7);
    uint32_t aux = 0, aux2 = 0, tail_node = 0;
    if (EXT) {
        aux = __ldg(c.edge_aux + e);
        aux2 = __ldg(c.edge_aux + (last ? e : e2));
        if (flags & OWNS) tail_node = __ldg(c.edge_from + e);
    }

    // 2a
    float v0 = v0m * E.vlim;
    if (EXT) v0 = fminf(v0, p.t_vmax[ty]);
    const int C = E.len;
    const float Cf = (float)C;
    const uint32_t lanes = edge_lanes(E), lanes2 = edge_lanes(E2);
    const uint32_t l2 = l < lanes2 - 1 ? l : lanes2 - 1;
    const uint32_t ctrl = edge_ctrl(E);
    bool may_cross, stop_node = false;
    if (!EXT) may_cross = last || ctrl != CTRL_SIGNAL || signal_green(E, k);
    else {
        may_cross = true;
        if (!last && (ctrl == CTRL_SIGNAL || ctrl == CTRL_SIGNAL_NM)) {
            // R35: movement (i, j) has phase number i*m + j; the host folded i*m*P into the offset, and
            // j*P (P = green + amber + allred in aux, j = rank of e2 among the outbound edges in aux2)
            // is taken off here -- added as cycle - j*P so that nothing goes negative
            uint32_t shift = 0;
            if (ctrl == CTRL_SIGNAL_NM) { const uint32_t jP = (aux2 >> 16) * (aux & 0xFFFFu); shift = jP ? (E.cyc_lc & 0xFFFFFFu) - jP : 0u; }
            const uint32_t pos = signal_pos(E, k, shift);
            may_cross = pos < (uint32_t)E.green;
            if (!may_cross && pos < (uint32_t)E.green + p.amber) {       // R36: amber
                const float rem = Cf - x;
                const float vv = v * v;
                const float need = p.two_b * rem;
                may_cross = vv > need;
            }
        } else if (!last && ctrl == CTRL_STOP) {
            // R34: the line stands as an obstacle until the vehicle has made its stop and the node is free
            const float rem = Cf - x;
            if (rem <= p.stop_dist && v <= p.stop_speed) flags |= STOPPED;
            stop_node = true;
            may_cross = (flags & STOPPED) != 0u;                         // and the node free: below
        }
    }
    const int lim = min(C - 1, ci + p.H);
    const int n_own = lim - ci;                        // cells c+1 .. min(C-1, c+H)
    const int Hp = p.H - (C - 1 - ci);
    bool want_next = !last && may_cross && Hp > 0;
    const int lim2 = min((int)E2.len - 1, Hp - 1);
    const uint32_t row2 = lane_row(E2, l2);

    // E5: the furthest this vehicle can get in one step; below the end of the edge it can neither
    // arrive nor cross, above it lanes are not changed (readings R12, R14)
    float reach = v + a_dt_i;
    reach = reach * p.dt;
    reach = x + reach;
    const bool may_leave = !(reach < Cf);
    bool lc_eval = false;
    uint32_t lt = l, rowt = row;
    if (p.lc_period != 0 && lanes >= 2 && !may_leave) {
        const int lti = (int)l + ((k & 1u) ? -1 : +1);
        const uint32_t turn = (k >> 1) + id;           // staggered: every lc_period-th pair of steps
        const bool my_turn = p.lc_pow2 ? (turn & (p.lc_period - 1u)) == 0u : turn % p.lc_period == 0u;
        if (lti >= 0 && lti < (int)lanes && x >= p.entry_zone_f && my_turn) {
            lc_eval = true;
            lt = (uint32_t)lti;
            rowt = lane_row(E, lt);
        }
    }
    const int lo = max(0, ci - p.Hb);

    // trip 3: next-edge window, target-lane windows and the cold part of the slot state
    uint4 sc = make_uint4(0, 0, 0, 0);
    if (may_leave || lc_eval) sc = ldcg4(S.C + slot);
    uint32_t free_from = 0;
    if (EXT && stop_node && may_cross) free_from = __ldcg(c.node_free_from + E.to_node);
    int cL = -1, cL2 = -1, cLt = -1, cF = -1;
    if (fast) {
        Win w_next, w_ta, w_tb;
        if (want_next) w_next = load_win(c.occ, row2, 0);
        if (lc_eval) { w_ta = load_win(c.occ, rowt, ci >> 7); w_tb = load_win(c.occ, rowt, ((ci - 1) >> 7) - 1); }
        if (EXT && stop_node) { may_cross = may_cross && free_from <= k; want_next = want_next && may_cross; }
        cL = first_occupied(w_own, ci + 1, n_own);                     // 2b
        if (cL < 0 && want_next) cL2 = first_occupied(w_next, 0, lim2 + 1);
        if (lc_eval) { cLt = first_occupied(w_ta, ci, lim - ci + 1); cF = last_occupied(w_tb, ci - 1, ci - lo); }
    } else {
        if (EXT && stop_node) { may_cross = may_cross && free_from <= k; want_next = want_next && may_cross; }
        cL = scan_ahead(c.occ, row, ci + 1, lim);
        if (cL < 0 && want_next) cL2 = scan_ahead(c.occ, row2, 0, lim2);
        if (lc_eval) { cLt = scan_ahead(c.occ, rowt, ci, lim); cF = scan_behind(c.occ, rowt, lo, ci - 1); }
    }

    // trip 4: speed codes (EXT: and types) of the vehicles found, and the route entry after the next edge
    uint32_t code_lead = 1, code_Lt = 1, code_F = 1, e3 = NONE32;
    uint32_t ty_lead = 0, ty_Lt = 0, ty_F = 0;
    if (cL >= 0) code_lead = code_at(c.codes, row, cL, p.cg);
    else if (cL2 >= 0) code_lead = code_at(c.codes, row2, cL2, p.cg);
    if (cLt >= 0) code_Lt = code_at(c.codes, rowt, cLt, p.cg);
    if (cF >= 0) code_F = code_at(c.codes, rowt, cF, p.cg);
    if (EXT && c.types) {
        if (cL >= 0) ty_lead = type_at(c.types, row, cL, p.cg);
        else if (cL2 >= 0) ty_lead = type_at(c.types, row2, cL2, p.cg);
        if (cLt >= 0) ty_Lt = type_at(c.types, rowt, cLt, p.cg);
        if (cF >= 0) ty_F = type_at(c.types, rowt, cF, p.cg);
    }
    if (may_leave && !last && sc.x + 2 < sc.y) e3 = __ldg(c.route_edges + sc.x + 2);

    // the code plane's granule holds ONE vehicle: a leader closer than a granule would share a code byte
    if (cL >= 0 && cL - ci < (1 << p.cg) && p.cg) atomicOr(&c.dyn->error, ERR_SPACING);

    // 2b gaps (E3): measured to the REAR of the vehicle ahead, i.e. with the leader's own length
    const float len_lead = EXT ? p.t_len[ty_lead & 3u] : p.len;
    const bool lead_on_edge = cL >= 0, has_lead = cL >= 0 || cL2 >= 0;
    float s_lead = 0.0f;
    if (lead_on_edge) {
        s_lead = (float)cL - len_lead;
        s_lead = s_lead - x;
    } else if (has_lead) {
        s_lead = Cf - x;
        s_lead = s_lead + (float)cL2;
        s_lead = s_lead - len_lead;
    }
    const float dv_lead = v - speed_decode(code_lead);

    // Eq. 7 against the own leader, the stop line and (below) the target lane: every evaluation is
    // spelled out unconditionally and the rule picks afterwards -- the chains are independent, so they
    // overlap instead of queueing behind one another's branches (the values are the same either way)
    const float fr = idm_free(v, v0);
    const float acc_free = a_i * fr;
    const float acc_follow = idm_follow(p, a_i, Kinv_i, fr, v, s_lead, dv_lead);
    const float acc_stop = idm_follow(p, a_i, Kinv_i, fr, v, Cf - x, v);             // 2c
    float acc = has_lead ? acc_follow : acc_free;
    if (!may_cross) acc = fminf(acc, acc_stop);

    // 2d gap acceptance G1-G3, then the mandatory rule or the MOBIL incentive G4
    bool accepted = false;
    const bool has_Lt = cLt >= 0;
    float s_Lt = 0.0f, at_c = 0.0f;
    if (lc_eval) {
        const float mand = __uint_as_float(sc.w);
        const bool has_F = cF >= 0;
        const float vLt = speed_decode(code_Lt), vF = speed_decode(code_F);
        const float len_Lt = EXT ? p.t_len[ty_Lt & 3u] : p.len;
        // the lag vehicle's acceleration ability and what is known of its desired speed (edge limit, type cap)
        const float a_F_ = EXT ? p.t_a[ty_F & 3u] : p.a, Kinv_F = EXT ? p.t_Kinv[ty_F & 3u] : p.Kinv;
        const float half_a_dt_F = EXT ? p.t_half_a_dt[ty_F & 3u] : p.half_a_dt;
        const float v0F = EXT ? fminf(E.vlim, p.t_vmax[ty_F & 3u]) : E.vlim;
        s_Lt = (float)cLt - len_Lt; s_Lt = s_Lt - x;                         // used only where has_Lt
        float s_lag = x - len_i; s_lag = s_lag - (float)(cF + 1);             // used only where has_F
        float m = (vF + 0.125f) + half_a_dt_F;                               // E4
        m = m * p.dt;
        float sF = (float)cLt - len_Lt;
        sF = sF - (float)(cF + 1);
        const float frF = idm_free(vF, v0F);
        const float aF_new = idm_follow(p, a_F_, Kinv_F, frF, vF, s_lag, vF - v);                       // G3
        const float a_F = has_Lt ? idm_follow(p, a_F_, Kinv_F, frF, vF, sF, vF - vLt) : a_F_ * frF;
        at_c = has_Lt ? idm_follow(p, a_i, Kinv_i, fr, v, s_Lt, v - vLt) : acc_free;
        const float a_c = lead_on_edge ? acc_follow : acc_free;
        const bool ok = (!has_Lt || s_Lt >= p.s0) &&                                                   // G1
                        (!has_F || (s_lag >= p.s0 && s_lag >= m && aF_new >= -p.b_safe));              // G2, G3
        const float rem = Cf - x;                                                                      // G4
        float inc = at_c - a_c;
        if (has_F) {
            float d2 = aF_new - a_F;
            d2 = p.politeness * d2;
            inc = inc + d2;
        }
        const bool inside = !last && rem <= mand;
        const bool mandatory = inside && l >= lanes2 && lt < l;
        const bool veto = inside && lt >= lanes2;
        accepted = ok && (mandatory || (!veto && inc > p.lc_threshold));
        if (!has_Lt) s_Lt = 0.0f;
    }

    // 2e integration (E2)
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

    // section 6.3.4: this vehicle's CO and fuel totals grow by rate * dt, with
    // the speed of state k and the acceleration just integrated (reading R30).  The pair travels
    // with the vehicle's slot: a plain read-modify-write, no atomics, reproducible.
    if (EMIS) {
        const float ar = (vt - v) * p.inv_dt;
        em.x = em.x + co_rate(v) * p.dt;
        em.y = em.y + fuel_rate(v, ar) * p.dt;
        __stcg(S.D + slot, em);
    }

    // 2f + the part of step 4 that concerns nobody else: this vehicle's own state k+1
    const uint32_t gc_from = (row << 7) + (uint32_t)ci;
    const uint32_t k1 = k + 1;
    // R34: a vehicle that holds the STOP node at the tail of its edge lets go once its rear bumper is
    // past it; the node is free from the next step on.  A reader of this step sees either the old
    // word (UINT32_MAX) or k+1 -- "held at step k" both ways.
    if (EXT && (flags & OWNS) && (xt >= len_i || xt >= Cf)) {
        __stcg(c.node_free_from + tail_node, k1);
        flags &= ~OWNS;
    }
    if (xt >= Cf) {
        if (!may_leave) atomicOr(&c.dyn->error, ERR_LOGIC);
        if (last) {                                    // ARRIVE: retires
            stcg4(S.A + slot, make_uint4(__float_as_uint(Cf), __float_as_uint(vt), row, l | flags));
            c.o_status[id] = 2; c.o_arrive[id] = k1; c.o_x[id] = Cf; c.o_v[id] = vt;
            c.o_edge[id] = e; c.o_lane[id] = (uint8_t)l; c.o_rpos[id] = sc.x;
            if (EMIS) c.emis[id] = em;                 // final totals, id-ordered
            atomicAdd(c.st_exited + e, 1u);
            atomicAdd(c.st_exit_steps + e, (unsigned long long)(k1 - sc.z));
            atomicAdd(&c.dyn->n_arrived, 1u);
            atomicAdd(&c.dyn->sum_arrive, (unsigned long long)k1);
            return make_uint4(gc_from, NONE32, 0, MR_CLEAR);
        }
        if (may_cross) {                               // CROSS: claims (one vehicle at a
            const unsigned long long w = claim_word(k, id);              // time; lowest id wins)
            const uint32_t g2 = E2.lane_base + l2;
            const bool node_claimed = ctrl == CTRL_PRIORITY || (EXT && ctrl == CTRL_STOP);
            const uint32_t h = node_claimed ? E.to_node : NONE32;
            atomicMin(c.lane_claim + g2, w);
            if (h != NONE32) atomicMin(c.node_claim + h, w);
            stcg4(S.A + slot, make_uint4(__float_as_uint(xt), __float_as_uint(vt), row, l | ALIVE | flags));
            float v0n = v0m * E2.vlim;
            if (EXT) v0n = fminf(v0n, p.t_vmax[ty]);
            stcg4(c.cr + 2 * (size_t)slot, make_uint4(row2, (uint32_t)E2.len | (l2 << 16), __float_as_uint(v0n), __float_as_uint(Cf)));
            stcg4(c.cr + 2 * (size_t)slot + 1, make_uint4(e3, (uint32_t)C, (EXT && ctrl == CTRL_STOP) ? 1u : 0u, 0));
            return make_uint4(gc_from, g2, h, MR_CROSS);
        }
        xt = Cf - 0.0625f; vt = 0.0f;                   // held at a red line (R17)
    }
    const uint32_t l_new = accepted ? lt : l, nrow = accepted ? rowt : row;
    const uint32_t code = speed_code(vt);
    stcg4(S.A + slot, make_uint4(__float_as_uint(xt), __float_as_uint(vt), nrow, l_new | ALIVE | flags));
    if (sample) {                                      // PAPER.md:437 one sample per minute
        atomicAdd(c.st_samp_cnt + e, 1u);
        atomicAdd(c.st_samp_code + e, (unsigned long long)(code - 1));
    }
    // a vehicle that keeps its cell and its speed code (a standing queue) leaves the atlas alone
    const uint32_t gc_to = (nrow << 7) + (uint32_t)(int)floorf(xt);
    if (gc_to == gc_from && code == speed_code(v)) return make_uint4(0, 0, 0, MR_NONE);
    return make_uint4(gc_from, gc_to, code | (ty << 8), MR_MOVE);
}

// DESIGN.md 2, step 3: the head of one departure queue.  A ready head takes
// a slot (kept as the queue's reservation until it wins) and writes its not-yet-alive state right
// away; phase 2 only flips it alive if it holds the lane claim.
__device__ __forceinline__ void departure_phase1(const Ctx& c, const Slots& S, uint32_t q, uint32_t k, const uint4 qr) {
    // qr = queue_rec[q] = { row, lane_base, end, edge }
    const uint4 qs = ldcg4(c.queue_state + q);         // { head, dep step of the head, reserved slot, - }
    uint4 cand = make_uint4(NONE32, 0, 0, 0);
    if (qs.x < qr.z && qs.y <= k) {
        const Win w = load_win(c.occ, qr.x, 0);
        const uint4 d0 = __ldg(c.dep_rec + 2 * (size_t)qs.x), d1 = __ldg(c.dep_rec + 2 * (size_t)qs.x + 1);
        uint32_t dep_next = NONE32;
        if (qs.x + 1 < qr.z) dep_next = __ldg(&c.dep_rec[2 * (size_t)(qs.x + 1) + 1].z);
        if (first_occupied(w, 0, (int)c.p.insert_clear) < 0) {
            uint32_t slot = qs.z;
            if (slot == NONE32) {
                slot = atomicAdd(&c.dyn->slot_alloc, 1u);
                if (slot < c.cap_slots) c.queue_state[q].z = slot;
            }
            if (slot >= c.cap_slots) atomicOr(&c.dyn->error, ERR_SLOTS);
            else {
                stcg4(S.A + slot, make_uint4(0u, 0u, qr.x, d1.w << TYPE_SHIFT));    // x = 0, v = 0, lane 0, its type, not alive
                stcg4(S.B + slot, make_uint4(qr.w, d1.y, d0.x, d0.y));
                stcg4(S.C + slot, make_uint4(d0.w, d1.x, k + 1, d0.z));
                if (S.D) __stcg(S.D + slot, make_float2(0.0f, 0.0f));
                atomicMin(c.lane_claim + qr.y, claim_word(k, d0.x));
                cand = make_uint4(d0.x, slot, qs.x, dep_next);
            }
        }
    }
    c.queue_cand[q] = cand;
}

// ------------------------------------------------------------------ phase 2

// Apply one move record; crossing vehicles resolve their claims first (step 4).
template <bool EXT>
__device__ __forceinline__ void vehicle_phase2(const Ctx& c, const Slots& S, uint32_t slot, uint32_t k,
                                               bool sample, const uint4 mr) {
    if (mr.w == MR_NONE) return;
    if (mr.w == MR_MOVE) {
        atlas_move(c, mr.x, mr.y, mr.z);
        if (EXT) atlas_set_type(c, mr.y, mr.z);
        return;
    }
    if (mr.w == MR_CLEAR) { atlas_vacate(c, mr.x); return; }
    // MR_CROSS: one trip for everything
    const uint4 sa = ldcg4(S.A + slot), sb = ldcg4(S.B + slot), sc = ldcg4(S.C + slot);
    const uint4 c0 = ldcg4(c.cr + 2 * (size_t)slot), c1 = ldcg4(c.cr + 2 * (size_t)slot + 1);
    // both claim words are fetched with the slot state, whether the node claim is needed or not:
    // a load issued only once `w` is known would be a second trip
    const unsigned long long wl = __ldcg(c.lane_claim + mr.y);
    const unsigned long long wn_raw = __ldcg(c.node_claim + (mr.z != NONE32 ? mr.z : 0u));
    const unsigned long long w = claim_word(k, sb.z);
    const unsigned long long wn = (mr.z != NONE32) ? wn_raw : w;
    const uint32_t e = sb.x, e2 = sb.y, l = sa.w & 0xFu, k1 = k + 1;
    uint32_t flags = EXT ? (sa.w & (TYPE_MASK | STOPPED | OWNS)) : 0u;
    float xn, vn;
    uint32_t gc_to, e_new;
    if (wl == w && wn == w) {                          // holds every claim it made: crosses
        if (EXT) {
            flags &= ~STOPPED;                         // the next STOP line wants a stop of its own
            if (c1.z) {                                // R34: it holds the node until its rear is past it
                __stcg(c.node_free_from + mr.z, 0xFFFFFFFFu);
                flags |= OWNS;
            }
        }
        const uint32_t len2 = c0.y & 0xFFFFu, l2 = c0.y >> 16;
        xn = __uint_as_float(sa.x) - __uint_as_float(c0.w);
        xn = fminf(xn, (float)len2 - 0.0625f);
        vn = fminf(__uint_as_float(sa.y), __uint_as_float(c0.z));       // R9
        stcg4(S.A + slot, make_uint4(__float_as_uint(xn), __float_as_uint(vn), c0.x, l2 | ALIVE | flags));
        stcg4(S.B + slot, make_uint4(e2, c1.x, sb.z, sb.w));
        stcg4(S.C + slot, make_uint4(sc.x + 1, sc.y, k1, sc.w));
        atomicAdd(c.st_entered + e2, 1u);
        atomicAdd(c.st_exited + e, 1u);
        atomicAdd(c.st_exit_steps + e, (unsigned long long)(k1 - sc.z));
        gc_to = (c0.x << 7) + (uint32_t)(int)floorf(xn);
        e_new = e2;
    } else {                                           // lost a claim: held at the line (R15)
        xn = __uint_as_float(c0.w) - 0.0625f; vn = 0.0f;
        stcg4(S.A + slot, make_uint4(__float_as_uint(xn), 0u, sa.z, l | ALIVE | flags));
        gc_to = (sa.z << 7) + (c1.y - 1u);
        e_new = e;
    }
    const uint32_t code = speed_code(vn);
    atlas_move(c, mr.x, gc_to, code);
    if (EXT) atlas_set_type(c, gc_to, (flags & TYPE_MASK) >> (TYPE_SHIFT - 8));
    if (sample) {
        atomicAdd(c.st_samp_cnt + e_new, 1u);
        atomicAdd(c.st_samp_code + e_new, (unsigned long long)(code - 1));
    }
}

// DESIGN.md 2, step 4 (departures): the winning queue head becomes ACTIVE at x = 0, v = 0, lane 0.
// `qr` = queue_rec[q]: static, kept in a register by the persistent kernel, so that the candidate
// and the claim word are ONE trip.
template <bool EXT>
__device__ __forceinline__ void departure_phase2(const Ctx& c, const Slots& S, uint32_t q, uint32_t k, bool sample,
                                                 const uint4 qr) {
    const uint4 cand = __ldcg(c.queue_cand + q);       // { id, slot, head, dep step of the next }
    const unsigned long long claim = __ldcg(c.lane_claim + qr.y);
    if (cand.x == NONE32) return;
    if (claim != claim_word(k, cand.x)) return;        // the slot stays reserved
    const uint32_t k1 = k + 1;
    uint32_t flags = 0;
    if (EXT) {                                         // its type was parked in the not-yet-alive record
        flags = __ldcg(&S.A[cand.y].w) & TYPE_MASK;
        atlas_set_type(c, qr.x << 7, flags >> (TYPE_SHIFT - 8));
    }
    stcg4(S.A + cand.y, make_uint4(0u, 0u, qr.x, ALIVE | flags));
    c.o_status[cand.x] = 1; c.o_insert[cand.x] = k1;
    c.queue_state[q] = make_uint4(cand.z + 1, cand.w, NONE32, 0);
    atlas_occupy(c, qr.x << 7, 1u);
    atomicAdd(c.st_entered + qr.w, 1u);
    atomicAdd(&c.dyn->n_departed, 1u);
    if (sample) atomicAdd(c.st_samp_cnt + qr.w, 1u);   // speed code - 1 == 0 at rest
}

// ------------------------------------------------------------------ phase drivers
// `mr_s`: this CTA's move records in shared memory, [mr_j][T]; slots beyond that use c.mr_g.

// `n_slots` must reach the threads without every warp of the grid loading the same word (one
// L2 slice would serve ~5000 requests in turn): one thread per CTA reads it, see the kernels.
template <bool EMIS, bool EXT>
__device__ __forceinline__ void phase1(const Ctx& c, const Slots& S, uint32_t k, const Who& me, uint4* mr_s,
                                       uint32_t mr_j, uint32_t n_slots, bool sample, uint32_t& n_upd, const uint4 qr0) {
    for (uint32_t j = 0;; j++) {
        const uint32_t s = me.slot(j);
        if (s >= n_slots) break;
        const uint4 mr = vehicle_phase1<EMIS, EXT>(c, S, s, k, sample, n_upd);
        if (j < mr_j) mr_s[j * me.T + me.t] = mr; else stcg4(c.mr_g + s, mr);
    }
    for (uint32_t j = 0;; j++) {
        const uint32_t q = me.qslot(j);
        if (q - (q & 31u) >= c.n_queues) break;
        if (q < c.n_queues) departure_phase1(c, S, q, k, j == 0 ? qr0 : __ldg(c.queue_rec + q));
    }
}

template <bool EXT>
__device__ __forceinline__ void phase2(const Ctx& c, const Slots& S, uint32_t k, const Who& me, const uint4* mr_s,
                                       uint32_t mr_j, uint32_t n_slots, bool sample, const uint4 qr0) {
    if (me.gtid() == 0) {
        // every slot handed out in phase 1 takes part from the next step on
        c.dyn->n_slots = min(__ldcg(&c.dyn->slot_alloc), c.cap_slots);
        c.dyn->k = k + 1;
        if (sample) c.dyn->n_samples = __ldcg(&c.dyn->n_samples) + 1;
    }
    for (uint32_t j = 0;; j++) {
        const uint32_t s = me.slot(j);
        if (s >= n_slots) break;
        const uint4 mr = (j < mr_j) ? mr_s[j * me.T + me.t] : ldcg4(c.mr_g + s);
        vehicle_phase2<EXT>(c, S, s, k, sample, mr);
    }
    for (uint32_t j = 0;; j++) {
        const uint32_t q = me.qslot(j);
        if (q - (q & 31u) >= c.n_queues) break;
        if (q < c.n_queues) departure_phase2<EXT>(c, S, q, k, sample, j == 0 ? qr0 : __ldg(c.queue_rec + q));
    }
}

// order-independent digest of state k+1 (test instrument, not on the timed path).
// `n_slots`: the slots of state k+1, read by one thread per CTA after the step's last barrier.
__device__ __forceinline__ void phase_digest(const Ctx& c, const Slots& S, unsigned long long* out, const Who& me,
                                             uint32_t n_slots) {
    unsigned long long sum = 0;
    for (uint32_t j = 0;; j++) {
        const uint32_t s = me.slot(j);
        if (s >= n_slots) break;
        const uint4 sa = ldcg4(S.A + s);
        if (!(sa.w & ALIVE)) continue;
        const uint4 sb = ldcg4(S.B + s);
        unsigned long long g = mix64((unsigned long long)sb.z);
        g = mix64(g ^ (((unsigned long long)sb.x << 8) | (sa.w & 0xFFu)));
        g = mix64(g ^ (((unsigned long long)sa.x << 32) | (unsigned long long)sa.y));
        sum += g;
    }
    if (me.gtid() == 0) {
        const uint32_t dep = __ldcg(&c.dyn->n_departed), arr = __ldcg(&c.dyn->n_arrived);
        unsigned long long g = mix64((unsigned long long)(c.V - dep));
        g = mix64(g ^ (unsigned long long)(dep - arr));
        g = mix64(g ^ (unsigned long long)arr);
        g = mix64(g ^ __ldcg(&c.dyn->sum_arrive));
        sum += g;
    }
    for (int o = 16; o; o >>= 1) sum += __shfl_xor_sync(0xFFFFFFFFu, sum, o);
    if ((threadIdx.x & 31) == 0 && sum) atomicAdd(out, sum);
}

}  // namespace ts
