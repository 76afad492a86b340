/*
 * ts_oracle.h -- ORACLE (test infrastructure, not product code).
 *
 * A plain, slow CPU restatement (single-threaded unless orc_set_threads is called) of the per-vehicle traffic
 * microsimulation of arxiv 1807.01148 (sections 6.3.2-6.3.3), following
 * SURVEY.md section 8(c) step by step (readings R1-R36 are listed in DESIGN.md; R27 fixes the
 * rounding order of two quotients inside Eq. 7; R31 vehicle types; R34-R36 the control
 * variants of PAPER.md:402).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may load this library.  It shares no code, header, table or helper with the CUDA path
 * under paper_1807_01148_b200/csrc/ and never includes include/trafficsim.h.
 *
 * Where the paper says the GPU method "represent[s] a road as a set of contiguous bytes"
 * and finds the leader by "check[ing] the following bytes", the oracle
 * deliberately does NOT build a byte map: it keeps an ordered list of vehicles per lane
 * ("a list of vehicles per lane", the structure the paper says it replaced) and applies
 * the same perception rule (cell index + quantised speed code).  orc_check() re-derives
 * every neighbour by an O(V^2) search over raw (edge, lane, x) as a second, independent
 * route to the same answer.
 *
 * Section 6.3.4 (Eq. 8 CO emission and Eq. 9 fuel consumption; SURVEY.md
 * section 8(f) row 2) is an optional pair of per-vehicle accumulators (readings R28-R30 in
 * DESIGN.md); it never feeds back into the traffic.  Pins: tests/test_oracle_emissions.py
 * (values of Eq. 8 / Eq. 9 at points worked by hand from the paper's coefficients, a standing
 * queue's idle totals, a cruising vehicle, and a fine-step fp64 quadrature of the lone-vehicle
 * acceleration run).
 *
 * Parity pins (tests/test_oracle_pins.py, test_oracle_invariants.py, test_oracle_scenarios.py,
 * test_oracle_lane_change_referee.py, test_oracle_variants.py):
 * P1 lone-vehicle closed form, P2 platoon equilibrium gap (on one edge, across nodes, behind a truck),
 * P3 standing queue, I1-I8 invariants, P4 brute force, P5 degenerate cases; a referee that re-derives
 * in fp64, from the rule text, EVERY lane-change decision of dense multi-lane scenarios (eligibility,
 * G1, G2 with its kinematic bound, G3, the mandatory rule at the first eligible turn, the veto of a
 * discretionary move into a lane that ends, the MOBIL incentive with the politeness term deciding both
 * ways) and is shown to catch the mutations a reviewer would try (dropped `m` term, flipped b_safe
 * sign, dropped politeness, `>=` -> `>`, dropped `+cL2`, `cF+1` -> `cF`); hold-at-line after a lost
 * claim; departure order and entry clearance; vehicle types (P1/P2 with the truck's own a, length and
 * cap; bodies never overlap); STOP control, n*m phases and amber checked from the recorded states
 * against the rule text and explicit timetables.  No sub-rule of vehicle_intent() is left pinned
 * oracle<->GPU only; what the PAPER does not fix (the readings R1-R44) is listed in DESIGN.md.
 * orc_set_threads: the intent loop may run on several host threads (results identical, tested);
 * the default and bench.py's cpu_baseline are single-threaded.
 */
#ifndef TS_ORACLE_H
#define TS_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Model parameters (PAPER.md:390 dt; :394-397 IDM a,b,T,s0; :399-400 lane change). */
typedef struct orc_params {
    float dt;            /* time step, s (0.5) */
    float a;             /* IDM acceleration ability, m/s^2 */
    float b;             /* IDM comfortable braking, m/s^2 */
    float T;             /* IDM desired time headway, s */
    float s0;            /* IDM minimum following distance, m */
    float veh_len;       /* vehicle length, m */
    float b_safe;        /* gap acceptance: max braking imposed on the new follower */
    float politeness;    /* MOBIL politeness p */
    float lc_threshold;  /* MOBIL incentive threshold, m/s^2 */
    float mand_dist_default; /* used where mand_dist_m == NULL */
    uint32_t lookahead_cells;     /* H  */
    uint32_t lookback_cells;      /* Hb */
    uint32_t lc_period;           /* 0 = lane changes disabled */
    uint32_t entry_zone_cells;
    uint32_t insert_clear_cells;
    uint32_t sample_period_steps; /* 0 = no sampling */
    uint32_t emissions;           /* non-zero: per-vehicle CO and fuel accumulators */
    /* Vehicle types ("a second type of vehicle to represent trucks, to reflect their
     * differences in size, acceleration, and maximum speed"; reading R31).  n_types == 0: one type
     * {veh_len, a, no speed cap}.  Otherwise type t = {type_len[t], type_a[t], type_vmax[t]} and
     * veh_len / a above are not used. */
    uint32_t n_types;             /* 0..4 */
    float type_len[4];            /* m */
    float type_a[4];              /* m/s^2 */
    float type_vmax[4];           /* m/s; desired speed = min(v0_mult * edge limit, type_vmax) */
    /* Control variants (readings R34-R36) */
    uint32_t amber_steps;         /* amber after every green (0 = none) */
    float stop_dist;              /* CTRL_STOP: a vehicle has made its stop once it is within stop_dist m */
    float stop_speed;             /*            of the line at no more than stop_speed m/s */
} orc_params;

/* Work counters: what a byte-scan method would have to touch. */
typedef struct orc_counters {
    uint64_t updates;          /* ACTIVE vehicle advanced one step */
    uint64_t own_cells;        /* cells between a vehicle and its leader / scan limit, own edge */
    uint64_t next_cells;       /* same, on the next route edge */
    uint64_t lc_evals;         /* lane-change evaluations */
    uint64_t lc_cells;         /* target-lane cells (ahead + behind) examined */
    uint64_t lc_accepts;
    uint64_t lc_mandatory;
    uint64_t crossings;        /* winning edge transitions */
    uint64_t cross_lost;       /* CROSS intents that lost a claim */
    uint64_t held_red;         /* held at a red stop line */
    uint64_t cap_bound;        /* advance limited by the no-overlap cap */
    uint64_t departures;
    uint64_t arrivals;
    uint64_t peak_active;
    /* the same scans counted in 16-cell pieces (a scan of n cells touches ceil(n/16) of them):
     * SURVEY.md 8(d) asks for the algorithmic bytes "rounded up to 16-cell chunks" beside the raw cells */
    uint64_t own_chunks16, next_chunks16, lc_chunks16;
} orc_counters;

typedef struct orc_sim orc_sim;

/* All pointers are host arrays owned by the caller and copied.  v0_mult / mand_dist_m / veh_type
 * may be NULL (veh_type: everybody is of type 0).  node_ctrl: 0 FREE, 1 PRIORITY, 2 SIGNAL (one
 * phase per inbound edge, R16), 3 STOP (R34), 4 SIGNAL_NM (one phase per movement, R35).  Returns NULL on invalid input (message in orc_last_error()). */
orc_sim *orc_create(uint32_t n_nodes, uint32_t n_edges,
                    const uint32_t *edge_from, const uint32_t *edge_to,
                    const uint32_t *edge_len_m, const uint8_t *edge_lanes,
                    const float *edge_vlim, const uint8_t *node_ctrl,
                    const uint32_t *sig_green_steps, const uint32_t *sig_allred_steps,
                    const uint32_t *sig_offset_steps,
                    uint32_t n_vehicles, const uint64_t *route_off,
                    const uint32_t *route_edges, const float *depart_time_s,
                    const float *v0_mult, const float *mand_dist_m, const uint8_t *veh_type,
                    const orc_params *params);

/* Advance n steps.  digests (nullable) receives one 64-bit digest per step (state k+1).
 * check: 0 none, 1 invariants I1-I7 every step, 2 additionally the O(V^2) brute-force
 * neighbour search (P4).  order_seed != 0 permutes the vehicle iteration order (I8).
 * Returns 0, or -1 on an invariant violation (message in orc_last_error()). */
int orc_step(orc_sim *s, uint32_t n, uint64_t *digests, int check, uint64_t order_seed);

/* Length-V arrays in vehicle-id order; any pointer may be NULL. */
void orc_read_state(const orc_sim *s, uint8_t *status, uint32_t *edge, uint8_t *lane,
                    uint32_t *cell, float *x, float *v, uint32_t *route_idx,
                    uint32_t *insert_step, uint32_t *arrive_step,
                    uint64_t *step, uint32_t *n_pending, uint32_t *n_active,
                    uint32_t *n_arrived);

/* Length-E arrays; any pointer may be NULL. */
void orc_read_edge_stats(orc_sim *s, uint32_t *entered, uint32_t *exited,
                         uint64_t *exit_steps_sum, uint32_t *sample_count_sum,
                         uint64_t *sample_speedcode_sum, uint32_t *n_samples, int reset);

/* Per-vehicle totals since step 0, length-V arrays in vehicle-id order (PAPER.md:408-423,
 * section 6.3.4): grams of CO (Eq. 8) and millilitres of fuel (Eq. 9).  Zeros unless
 * orc_params.emissions was set.  Either pointer may be NULL. */
void orc_read_emissions(const orc_sim *s, float *co_g, float *fuel_ml);

/* Eq. 8 and Eq. 9 as the simulator evaluates them (fp32): CO rate in g/s at speed v (m/s);
 * fuel rate in mL/s at speed v and acceleration acc (m/s^2). */
float orc_co_rate(float v);
float orc_fuel_rate(float v, float acc);

void orc_get_counters(const orc_sim *s, orc_counters *out);

/* Host threads for the intent loop of step 2 (default 1 = the plain sequential program).
 * Every intent reads state k only and writes only its own vehicle's intent, so the loop's
 * iterations are independent; results are identical for every n (tests/test_oracle_invariants.py).
 * Exists so that tests/golden/make_golden.py can get through the whole run of config 4
 * (5.4e10 vehicle-updates); bench.py's cpu_baseline times the default. */
void orc_set_threads(orc_sim *s, int n);
void orc_destroy(orc_sim *s);
const char *orc_last_error(void);

/* Scalar building blocks exported so the pins can probe them directly. */
float orc_idm(const orc_params *p, float v, float v0, int has_leader, float s, float dv);
uint8_t orc_speed_code(float v);
float orc_speed_decode(uint8_t code);
int orc_signal_green(uint32_t green, uint32_t allred, uint32_t offset, uint32_t n_in,
                     uint32_t in_rank, uint64_t k);
/* 0 red, 1 green, 2 amber; n_out == 0: one phase per inbound edge, else one per movement. */
int orc_signal_phase(uint32_t green, uint32_t amber, uint32_t allred, uint32_t offset, uint32_t n_in,
                     uint32_t n_out, uint32_t in_rank, uint32_t out_rank, uint64_t k);
uint64_t orc_mix64(uint64_t z);

#ifdef __cplusplus
}
#endif
#endif
