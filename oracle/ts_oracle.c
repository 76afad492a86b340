/*
 * ts_oracle.c -- ORACLE (test infrastructure, not product code).  See ts_oracle.h.
 *
 * Build: gcc -std=c99 -O2 -ffp-contract=off -fno-fast-math -fPIC -shared (oracle/build.py).
 * All model arithmetic is fp32, one rounding per written operation, no fused multiply-add
 * (SURVEY.md 8(c) "Arithmetic"; reading R21).  Each expression below is spelled
 * as a sequence of single operations on `float` temporaries for that reason.
 *
 * Vocabulary follows the paper: edge, lane, vehicle, leader ("the leading car",
 * PAPER.md:406), lead/lag gap, s, s0, T, a, b, v0 (Eq. 7).
 */
#include "ts_oracle.h"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { ST_PENDING = 0, ST_ACTIVE = 1, ST_ARRIVED = 2 };
enum { CTRL_FREE = 0, CTRL_PRIORITY = 1, CTRL_SIGNAL = 2, CTRL_STOP = 3, CTRL_SIGNAL_NM = 4 };
enum { SIG_RED = 0, SIG_GREEN = 1, SIG_AMBER = 2 };
#define MAX_TYPES 4
enum { ACT_STAY = 0, ACT_ARRIVE = 1, ACT_CROSS = 2 };
#define NONE (-1)
#define NO_CLAIM 0xFFFFFFFFu

static char g_err[512];
const char *orc_last_error(void) { return g_err; }
#define FAIL(...) do { snprintf(g_err, sizeof g_err, __VA_ARGS__); } while (0)

struct orc_sim {
    orc_params p;
    /* per vehicle type ("a second type of vehicle to represent trucks ... size,
     * acceleration, and maximum speed"; reading R31): length, acceleration ability a, 1/(2 sqrt(a b))
     * (fp32, computed once, reading R27), speed cap */
    uint32_t n_types;
    float t_len[MAX_TYPES], t_a[MAX_TYPES], t_Kinv[MAX_TYPES], t_vmax[MAX_TYPES];
    float two_b;                   /* 2*b, fp32, computed once (amber rule, reading R36) */
    uint8_t *veh_type;             /* [V] */
    uint32_t N, E, V;
    /* network */
    uint32_t *edge_from, *edge_to, *edge_len;
    uint8_t *edge_lanes, *edge_in_rank, *edge_out_rank;
    float *edge_vlim;
    uint8_t *node_ctrl;
    uint32_t *node_n_in, *node_n_out, *sig_green, *sig_allred, *sig_offset;
    /* CTRL_STOP (reading R34): first step at which the node is free again; UINT32_MAX while a
     * vehicle that crossed it has not yet cleared it with its rear bumper */
    uint32_t *node_free_from;
    uint8_t *made_stop, *owns_node; /* [V] has come to a halt at the stop line of its edge / holds the node at its edge's tail */
    uint8_t *stop_t;               /* [V] intent: made_stop after this step */
    uint64_t *lane_base;           /* [E+1] global lane index of (e,0) */
    /* demand */
    uint64_t *route_off;
    uint32_t *route_edges;
    uint32_t *dep_step;            /* [V] ceil(depart_time/dt), double arithmetic */
    float *v0_mult, *mand_dist;
    /* per-origin-edge FIFO queues of pending vehicles, ordered by (dep_step, id) */
    uint32_t n_queues;
    uint32_t *queue_edge;          /* [n_queues] */
    uint64_t *queue_off;           /* [n_queues+1] into queue_veh */
    uint64_t *queue_head;          /* [n_queues] next pending position */
    uint32_t *queue_veh;           /* [V] */
    /* vehicle state at step k */
    uint8_t *status, *lane;
    uint32_t *r, *edge, *insert_step, *arrive_step, *enter_step;
    float *x, *v;
    /* per-lane ordered lists: ahead = next vehicle in driving direction */
    int32_t *ahead, *behind;       /* [V] */
    int32_t *lane_head, *lane_tail;/* [n_lanes] front-most / rear-most vehicle */
    /* active set (iteration order is irrelevant: I8) */
    uint32_t *active; uint32_t n_active_list; uint32_t *active_pos;
    /* intents of the current step */
    float *xt, *vt;
    uint8_t *act, *ln, *l2;
    uint32_t *e2;
    /* claims (minimum id) with touched lists so that nothing is cleared wholesale */
    uint32_t *lane_claim, *node_claim;
    uint64_t *touched_lanes; uint64_t n_touched_lanes;
    uint32_t *touched_nodes; uint32_t n_touched_nodes;
    uint32_t *dep_cand;            /* [n_queues] vehicle claiming a departure this step or NO_CLAIM */
    /* relink work lists */
    uint32_t *relink; uint32_t n_relink;
    uint64_t *entry_lane; uint32_t *cross_node; uint32_t n_entry, n_cross_node; /* I7 bookkeeping (check mode) */
    /* outputs */
    uint32_t *entered, *exited, *sample_count_sum;
    uint64_t *exit_steps_sum, *sample_speedcode_sum;
    float *co_g, *fuel_ml;         /* [V] section 6.3.4 accumulators */
    uint32_t n_samples;
    uint64_t k;                    /* current step */
    uint32_t n_pending, n_active, n_arrived;
    uint64_t sum_arrive_step;
    orc_counters cnt;
    int threads;                   /* host threads for the intent loop of step 2 (orc_set_threads) */
};

/* ---------------------------------------------------------------- scalar building blocks */

/* Perception (reading R5): a vehicle is visible to others only as its cell and a
 * speed code at 0.25 m/s resolution; 0 means "empty", so codes start at 1. */
uint8_t orc_speed_code(float v) {
    float q = v * 4.0f;
    q = q + 0.5f;
    int c = (int)q;
    if (c > 254) c = 254;
    return (uint8_t)(1 + c);
}
float orc_speed_decode(uint8_t code) { return (float)((int)code - 1) * 0.25f; }

/* Intelligent Driver Model, Eq. 7 (readings R1, R2, R8):
 *   dv/dt = a * ( 1 - (v/v0)^4 - ((s0 + max(0, T v + v dv / (2 sqrt(a b)))) / max(s, 0.5))^2 )
 * with s the net gap to the car ahead and dv = v - v_leader.
 * Reading R27: the two quotients whose divisor does not depend on the traffic are
 * formed with a reciprocal rounded once -- v/v0 as v * (1/v0), v dv/(2 sqrt(ab)) as (v dv) * (1/K)
 * -- each still one rounding per written operation; s* / s stays a division. */
static float idm(const orc_sim *S, uint32_t ty, float v, float v0, int has, float s, float dv) {
    const orc_params *p = &S->p;
    const float a = S->t_a[ty];        /* "a is the acceleration ability of the vehicle" */
    float rinv = 1.0f / v0;
    float r = v * rinv;
    float r2 = r * r;
    float r4 = r2 * r2;
    float fr = 1.0f - r4;
    if (!has) return a * fr;
    float t = v * p->T;
    float u = v * dv;
    float w = u * S->t_Kinv[ty];
    t = t + w;
    t = fmaxf(t, 0.0f);
    float ss = p->s0 + t;
    float se = fmaxf(s, 0.5f);
    float q = ss / se;
    float q2 = q * q;
    float d = fr - q2;
    return a * d;
}

float orc_idm(const orc_params *p, float v, float v0, int has_leader, float s, float dv) {
    orc_sim tmp;
    tmp.p = *p;
    float ab = p->a * p->b;
    { float K = 2.0f * sqrtf(ab); tmp.t_Kinv[0] = 1.0f / K; tmp.t_a[0] = p->a; }
    return idm(&tmp, 0, v, v0, has_leader, s, dv);
}

/* CO emission rate, Eq. 8 (Stein and Walker 2003):
 *   P = -0.064 + 0.0056 v_m + 0.00026 (v_m - 50)^2      [g/s], v_m = speed in miles per hour.
 * v is in m/s; 1 m/s = 3600/1609.344 mph = 2.2369363 mph (reading R28: the fp32 nearest to that
 * ratio).  Evaluated left to right, one rounding per written operation. */
float orc_co_rate(float v) {
    float vm = v * 2.2369363f;
    float P = 0.0056f * vm;
    P = -0.064f + P;
    float d = vm - 50.0f;
    float d2 = d * d;
    float q = 0.00026f * d2;
    P = P + q;
    return P;
}

/* Fuel consumption rate, Eq. 9 (Akcelik 1989):
 *   f = 0.666 + 0.072 (0.269 v + 0.0171 v^2 + 0.000672 v^3 + 1.680 a v + P_ea)   [mL/s],
 *   P_ea = 0.79296 a^2 v for a > 0 (else 0), v in m/s, a in m/s^2.
 * Reading R29: the bracket (the tractive power demand) is floored at 0, so a braking vehicle
 * burns the idle rate 0.666 mL/s and never a negative amount -- the paper prints no floor, the
 * model it cites has one.  Terms are added in the printed order. */
float orc_fuel_rate(float v, float acc) {
    float v2 = v * v;
    float v3 = v2 * v;
    float g = 0.269f * v;
    float h = 0.0171f * v2;
    g = g + h;
    h = 0.000672f * v3;
    g = g + h;
    h = 1.680f * acc;
    h = h * v;
    g = g + h;
    if (acc > 0.0f) {
        h = acc * acc;
        h = 0.79296f * h;
        h = h * v;
        g = g + h;
    }
    g = fmaxf(g, 0.0f);
    float f = 0.072f * g;
    f = 0.666f + f;
    return f;
}

/* Fixed-time signal, one protected phase per inbound edge in round robin
 * ("round robin"; reading R16). */
int orc_signal_green(uint32_t green, uint32_t allred, uint32_t offset, uint32_t n_in,
                     uint32_t in_rank, uint64_t k) {
    uint64_t P = (uint64_t)green + allred;
    uint64_t cyc = (uint64_t)n_in * P;
    uint64_t t = (k + offset) % cyc;
    return (t / P == in_rank) && (t % P < green);
}

/* The same plan with an amber interval after the green (reading R36) and, for n_out > 0, the
 * paper's literal phasing ("given an intersection with n inbound edges and m outbound,
 * our system creates the geometric combination nm of necessary traffic phasing ... in a round robing
 * logic"; reading R35): one phase per MOVEMENT (inbound edge i, outbound edge j), in the order
 * i*m + j, each green + amber + allred steps long.  n_out == 0: one phase per inbound edge (R16). */
int orc_signal_phase(uint32_t green, uint32_t amber, uint32_t allred, uint32_t offset, uint32_t n_in,
                     uint32_t n_out, uint32_t in_rank, uint32_t out_rank, uint64_t k) {
    uint64_t P = (uint64_t)green + amber + allred;
    uint64_t n_phases = n_out ? (uint64_t)n_in * n_out : n_in;
    uint64_t mine = n_out ? (uint64_t)in_rank * n_out + out_rank : in_rank;
    uint64_t t = (k + offset) % (n_phases * P);
    if (t / P != mine) return SIG_RED;
    uint64_t pos = t % P;
    if (pos < green) return SIG_GREEN;
    if (pos < (uint64_t)green + amber) return SIG_AMBER;
    return SIG_RED;
}

/* SplitMix64 finaliser. */
uint64_t orc_mix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

static uint32_t fbits(float f) { uint32_t u; memcpy(&u, &f, 4); return u; }

/* ---------------------------------------------------------------- construction */

static void *xcalloc(size_t n, size_t sz) {
    void *p = calloc(n ? n : 1, sz);
    if (!p) { fprintf(stderr, "oracle: out of memory\n"); abort(); }
    return p;
}
static void *xdup(const void *src, size_t n, size_t sz) {
    void *p = xcalloc(n, sz);
    if (n) memcpy(p, src, n * sz);
    return p;
}

typedef struct { uint32_t edge, dep, id; } qkey;
static int qkey_cmp(const void *a, const void *b) {
    const qkey *x = (const qkey *)a, *y = (const qkey *)b;
    if (x->edge != y->edge) return x->edge < y->edge ? -1 : 1;
    if (x->dep != y->dep) return x->dep < y->dep ? -1 : 1;
    if (x->id != y->id) return x->id < y->id ? -1 : 1;
    return 0;
}

orc_sim *orc_create(uint32_t n_nodes, uint32_t n_edges,
                    const uint32_t *edge_from, const uint32_t *edge_to,
                    const uint32_t *edge_len_m, const uint8_t *edge_lanes,
                    const float *edge_vlim, const uint8_t *node_ctrl,
                    const uint32_t *sig_green_steps, const uint32_t *sig_allred_steps,
                    const uint32_t *sig_offset_steps,
                    uint32_t n_vehicles, const uint64_t *route_off,
                    const uint32_t *route_edges, const float *depart_time_s,
                    const float *v0_mult, const float *mand_dist_m, const uint8_t *veh_type,
                    const orc_params *params) {
    const orc_params *p = params;
    g_err[0] = 0;
    if (!(p->dt > 0) || !(p->a > 0) || !(p->b > 0) || !(p->T >= 0) || !(p->s0 >= 0) ||
        !(p->veh_len >= 2.0f) || p->lookahead_cells == 0 || p->lookahead_cells % 16 ||
        p->insert_clear_cells == 0 || p->insert_clear_cells > 16 || p->n_types > MAX_TYPES) {
        FAIL("bad params"); return NULL;
    }
    /* vehicle types (reading R31): none given = one type {veh_len, a, no speed cap} */
    uint32_t n_types = p->n_types ? p->n_types : 1;
    float max_len = 0.0f, max_a = 0.0f;
    for (uint32_t t = 0; t < n_types; t++) {
        float len_t = p->n_types ? p->type_len[t] : p->veh_len;
        float a_t = p->n_types ? p->type_a[t] : p->a;
        float vmax_t = p->n_types ? p->type_vmax[t] : INFINITY;
        if (!(len_t >= 2.0f) || !(a_t > 0) || !(vmax_t > 0)) { FAIL("vehicle type %u", t); return NULL; }
        if (len_t > max_len) max_len = len_t;
        if (a_t > max_a) max_a = a_t;
    }
    float max_mult = 1.0f;
    for (uint32_t i = 0; i < n_vehicles; i++) {
        if (v0_mult) {
            if (!(v0_mult[i] > 0)) { FAIL("v0_mult[%u] <= 0", i); return NULL; }
            if (v0_mult[i] > max_mult) max_mult = v0_mult[i];
        }
        if (!(depart_time_s[i] >= 0)) { FAIL("depart_time_s[%u] < 0", i); return NULL; }
        if (route_off[i + 1] <= route_off[i]) { FAIL("route %u empty", i); return NULL; }
        if (veh_type && veh_type[i] >= n_types) { FAIL("veh_type[%u]", i); return NULL; }
    }
    float max_vlim = 0.0f;
    for (uint32_t e = 0; e < n_edges; e++) {
        if (edge_vlim[e] > max_vlim) max_vlim = edge_vlim[e];
        if (edge_from[e] >= n_nodes || edge_to[e] >= n_nodes) { FAIL("edge %u endpoint", e); return NULL; }
        if (edge_len_m[e] < 16 || edge_len_m[e] > 65535) { FAIL("edge %u length", e); return NULL; }
        if (edge_lanes[e] < 1 || edge_lanes[e] > 8) { FAIL("edge %u lanes", e); return NULL; }
        if (!(edge_vlim[e] > 0)) { FAIL("edge %u vlim", e); return NULL; }
        /* a vehicle entering an edge must land short of the zone where lanes may be changed */
        double adv = (double)edge_vlim[e] * max_mult * p->dt + 0.5 * max_a * p->dt * p->dt + max_len;
        if (!(adv < (double)p->entry_zone_cells)) { FAIL("edge %u: entry zone too short", e); return NULL; }
    }
    {   /* the look-ahead (and the look-back of the lane-change rule) must reach further than a
         * vehicle can advance in one step plus a vehicle length: nobody jumps over a leader unseen */
        double adv = (double)max_vlim * max_mult * p->dt + 0.5 * max_a * p->dt * p->dt + max_len;
        if (!((double)p->lookahead_cells >= adv)) { FAIL("lookahead_cells too short"); return NULL; }
        if (p->lc_period != 0 && !((double)p->lookback_cells >= adv)) { FAIL("lookback_cells too short"); return NULL; }
    }
    int any_stop = 0;
    for (uint32_t h = 0; h < n_nodes; h++) {
        if (node_ctrl[h] > CTRL_SIGNAL_NM) { FAIL("node %u ctrl", h); return NULL; }
        if ((node_ctrl[h] == CTRL_SIGNAL || node_ctrl[h] == CTRL_SIGNAL_NM) && sig_green_steps[h] == 0) { FAIL("node %u green", h); return NULL; }
        if (node_ctrl[h] == CTRL_STOP) any_stop = 1;
    }
    /* a vehicle that holds a STOP node lets go once its rear bumper is past it, on the edge it entered */
    if (any_stop && !(max_len < 16.0f)) { FAIL("STOP control needs vehicle lengths < 16 m"); return NULL; }
    for (uint32_t i = 0; i < n_vehicles; i++)
        for (uint64_t j = route_off[i]; j < route_off[i + 1]; j++) {
            if (route_edges[j] >= n_edges) { FAIL("route %u edge id", i); return NULL; }
            if (j > route_off[i] && edge_to[route_edges[j - 1]] != edge_from[route_edges[j]]) {
                FAIL("route %u not contiguous", i); return NULL;
            }
        }

    orc_sim *S = (orc_sim *)xcalloc(1, sizeof *S);
    S->p = *p;
    S->n_types = n_types;
    for (uint32_t t = 0; t < n_types; t++) {
        S->t_len[t] = p->n_types ? p->type_len[t] : p->veh_len;
        S->t_a[t] = p->n_types ? p->type_a[t] : p->a;
        S->t_vmax[t] = p->n_types ? p->type_vmax[t] : INFINITY;
        float ab = S->t_a[t] * p->b; float K = 2.0f * sqrtf(ab); S->t_Kinv[t] = 1.0f / K;
    }
    S->two_b = 2.0f * p->b;
    S->N = n_nodes; S->E = n_edges; S->V = n_vehicles;
    uint32_t N = n_nodes, E = n_edges, V = n_vehicles;
    S->edge_from = xdup(edge_from, E, 4); S->edge_to = xdup(edge_to, E, 4);
    S->edge_len = xdup(edge_len_m, E, 4); S->edge_lanes = xdup(edge_lanes, E, 1);
    S->edge_vlim = xdup(edge_vlim, E, 4); S->node_ctrl = xdup(node_ctrl, N, 1);
    S->sig_green = xdup(sig_green_steps, N, 4); S->sig_allred = xdup(sig_allred_steps, N, 4);
    S->sig_offset = xdup(sig_offset_steps, N, 4);
    /* in_rank: rank of e among the inbound edges of its head node, by edge index */
    S->node_n_in = xcalloc(N, 4); S->edge_in_rank = xcalloc(E, 1);
    S->node_n_out = xcalloc(N, 4); S->edge_out_rank = xcalloc(E, 1);
    for (uint32_t e = 0; e < E; e++) {
        uint32_t h = edge_to[e], t = edge_from[e];
        if (S->node_n_in[h] >= 255) { FAIL("node %u in-degree", h); orc_destroy(S); return NULL; }
        S->edge_in_rank[e] = (uint8_t)S->node_n_in[h]++;
        if (S->node_n_out[t] >= 255) { FAIL("node %u out-degree", t); orc_destroy(S); return NULL; }
        S->edge_out_rank[e] = (uint8_t)S->node_n_out[t]++;   /* rank among the outbound edges, by edge index */
    }
    S->node_free_from = xcalloc(N, 4);
    S->made_stop = xcalloc(V, 1); S->owns_node = xcalloc(V, 1); S->stop_t = xcalloc(V, 1);
    S->veh_type = xcalloc(V, 1);
    if (veh_type) memcpy(S->veh_type, veh_type, V);
    S->lane_base = xcalloc((size_t)E + 1, 8);
    for (uint32_t e = 0; e < E; e++) S->lane_base[e + 1] = S->lane_base[e] + edge_lanes[e];
    uint64_t n_lanes = S->lane_base[E];

    S->route_off = xdup(route_off, (size_t)V + 1, 8);
    S->route_edges = xdup(route_edges, route_off[V], 4);
    S->dep_step = xcalloc(V, 4); S->v0_mult = xcalloc(V, 4); S->mand_dist = xcalloc(V, 4);
    for (uint32_t i = 0; i < V; i++) {
        S->dep_step[i] = (uint32_t)ceil((double)depart_time_s[i] / (double)p->dt);
        S->v0_mult[i] = v0_mult ? v0_mult[i] : 1.0f;
        S->mand_dist[i] = mand_dist_m ? mand_dist_m[i] : p->mand_dist_default;
    }
    /* departure queues: one per distinct first edge, FIFO by (dep_step, id) (reading R19) */
    qkey *keys = xcalloc(V, sizeof *keys);
    for (uint32_t i = 0; i < V; i++) {
        keys[i].edge = route_edges[route_off[i]]; keys[i].dep = S->dep_step[i]; keys[i].id = i;
    }
    qsort(keys, V, sizeof *keys, qkey_cmp);
    uint32_t nq = 0;
    for (uint32_t i = 0; i < V; i++) if (i == 0 || keys[i].edge != keys[i - 1].edge) nq++;
    S->n_queues = nq;
    S->queue_edge = xcalloc(nq, 4); S->queue_off = xcalloc((size_t)nq + 1, 8);
    S->queue_head = xcalloc(nq, 8); S->queue_veh = xcalloc(V, 4); S->dep_cand = xcalloc(nq, 4);
    uint32_t q = 0;
    for (uint32_t i = 0; i < V; i++) {
        if (i == 0 || keys[i].edge != keys[i - 1].edge) { S->queue_edge[q] = keys[i].edge; S->queue_off[q] = i; q++; }
        S->queue_veh[i] = keys[i].id;
    }
    S->queue_off[nq] = V;
    for (q = 0; q < nq; q++) S->queue_head[q] = S->queue_off[q];
    free(keys);

    S->status = xcalloc(V, 1); S->lane = xcalloc(V, 1);
    S->r = xcalloc(V, 4); S->edge = xcalloc(V, 4); S->insert_step = xcalloc(V, 4);
    S->arrive_step = xcalloc(V, 4); S->enter_step = xcalloc(V, 4);
    S->x = xcalloc(V, 4); S->v = xcalloc(V, 4);
    S->ahead = xcalloc(V, 4); S->behind = xcalloc(V, 4);
    S->lane_head = xcalloc(n_lanes, 4); S->lane_tail = xcalloc(n_lanes, 4);
    for (uint64_t g = 0; g < n_lanes; g++) { S->lane_head[g] = NONE; S->lane_tail[g] = NONE; }
    for (uint32_t i = 0; i < V; i++) { S->ahead[i] = NONE; S->behind[i] = NONE; S->edge[i] = route_edges[route_off[i]]; }
    S->active = xcalloc(V, 4); S->active_pos = xcalloc(V, 4);
    S->xt = xcalloc(V, 4); S->vt = xcalloc(V, 4);
    S->act = xcalloc(V, 1); S->ln = xcalloc(V, 1); S->l2 = xcalloc(V, 1); S->e2 = xcalloc(V, 4);
    S->lane_claim = xcalloc(n_lanes, 4); S->node_claim = xcalloc(N, 4);
    for (uint64_t g = 0; g < n_lanes; g++) S->lane_claim[g] = NO_CLAIM;
    for (uint32_t h = 0; h < N; h++) S->node_claim[h] = NO_CLAIM;
    S->touched_lanes = xcalloc((size_t)V + nq, 8); S->touched_nodes = xcalloc(V, 4);
    S->relink = xcalloc(V, 4);
    S->entry_lane = xcalloc((size_t)V, 8); S->cross_node = xcalloc(V, 4);
    S->entered = xcalloc(E, 4); S->exited = xcalloc(E, 4); S->sample_count_sum = xcalloc(E, 4);
    S->exit_steps_sum = xcalloc(E, 8); S->sample_speedcode_sum = xcalloc(E, 8);
    S->co_g = xcalloc(V, 4); S->fuel_ml = xcalloc(V, 4);
    S->n_pending = V;
    S->threads = 1;
    return S;
}

void orc_destroy(orc_sim *S) {
    if (!S) return;
    free(S->edge_from); free(S->edge_to); free(S->edge_len); free(S->edge_lanes);
    free(S->edge_in_rank); free(S->edge_vlim); free(S->node_ctrl); free(S->node_n_in);
    free(S->sig_green); free(S->sig_allred); free(S->sig_offset); free(S->lane_base);
    free(S->route_off); free(S->route_edges); free(S->dep_step); free(S->v0_mult);
    free(S->mand_dist); free(S->queue_edge); free(S->queue_off); free(S->queue_head);
    free(S->queue_veh); free(S->dep_cand); free(S->status); free(S->lane); free(S->r);
    free(S->edge); free(S->insert_step); free(S->arrive_step); free(S->enter_step);
    free(S->x); free(S->v); free(S->ahead); free(S->behind); free(S->lane_head);
    free(S->lane_tail); free(S->active); free(S->active_pos); free(S->xt); free(S->vt);
    free(S->act); free(S->ln); free(S->l2); free(S->e2); free(S->lane_claim);
    free(S->node_claim); free(S->touched_lanes); free(S->touched_nodes); free(S->relink);
    free(S->entry_lane); free(S->cross_node);
    free(S->entered); free(S->exited); free(S->sample_count_sum); free(S->exit_steps_sum);
    free(S->sample_speedcode_sum); free(S->co_g); free(S->fuel_ml);
    free(S->node_n_out); free(S->edge_out_rank); free(S->node_free_from);
    free(S->made_stop); free(S->owns_node); free(S->stop_t); free(S->veh_type);
    free(S);
}

/* ---------------------------------------------------------------- one step: intent */

static int32_t cell_of(const orc_sim *S, uint32_t i) { return (int32_t)floorf(S->x[i]); }

static void claim_lane(orc_sim *S, uint64_t g, uint32_t id) {
    if (S->lane_claim[g] == NO_CLAIM) S->touched_lanes[S->n_touched_lanes++] = g;
    if (id < S->lane_claim[g]) S->lane_claim[g] = id;
}
static void claim_node(orc_sim *S, uint32_t h, uint32_t id) {
    if (S->node_claim[h] == NO_CLAIM) S->touched_nodes[S->n_touched_nodes++] = h;
    if (id < S->node_claim[h]) S->node_claim[h] = id;
}

/* Neighbours of position c in lane g of the current edge, from the ordered list:
 * *lead = rear-most vehicle with cell >= c_from, *lag = front-most vehicle with cell < c_from.
 * (The byte-scan method would find the same two by scanning the lane's bytes.) */
static void lane_neighbours(const orc_sim *S, uint64_t g, int32_t c_from, int32_t *lead, int32_t *lag) {
    int32_t j = S->lane_tail[g], prev = NONE;
    while (j != NONE && cell_of(S, (uint32_t)j) < c_from) { prev = j; j = S->ahead[j]; }
    *lead = j; *lag = prev;
}

/* intent of ACTIVE vehicle i from state k only. */
static void vehicle_intent(orc_sim *S, uint32_t i, orc_counters *cnt) {
    const orc_params *p = &S->p;
    const uint64_t k = S->k;
    const uint32_t e = S->edge[i];
    const uint32_t l = S->lane[i];
    const float x = S->x[i], v = S->v[i];
    const int32_t C = (int32_t)S->edge_len[e];
    const float Cf = (float)C;
    const int32_t H = (int32_t)p->lookahead_cells, Hb = (int32_t)p->lookback_cells;
    const uint32_t ty = S->veh_type[i];
    const float len = S->t_len[ty];             /* this vehicle's own length */
    const float a_i = S->t_a[ty];
    const uint32_t lanes_e = S->edge_lanes[e];

    /* 2a; a truck's desired speed is capped by its type's maximum (reading R31) */
    float v0 = S->v0_mult[i] * S->edge_vlim[e];
    v0 = fminf(v0, S->t_vmax[ty]);
    const uint64_t rpos = S->route_off[i] + S->r[i];
    const int last = (rpos + 1 == S->route_off[i + 1]);
    uint32_t e2 = 0, l2 = 0, lanes_e2 = 0;
    if (!last) {
        e2 = S->route_edges[rpos + 1];
        lanes_e2 = S->edge_lanes[e2];
        l2 = l < lanes_e2 - 1 ? l : lanes_e2 - 1;
    }
    const uint32_t h = S->edge_to[e];
    const uint32_t ctrl = S->node_ctrl[h];
    int may_cross = 1;
    uint8_t made_stop = S->made_stop[i];
    if (!last && (ctrl == CTRL_SIGNAL || ctrl == CTRL_SIGNAL_NM)) {
        int ph = orc_signal_phase(S->sig_green[h], p->amber_steps, S->sig_allred[h], S->sig_offset[h],
                                  S->node_n_in[h], ctrl == CTRL_SIGNAL_NM ? S->node_n_out[h] : 0,
                                  S->edge_in_rank[e], S->edge_out_rank[e2], k);
        may_cross = ph == SIG_GREEN;
        if (ph == SIG_AMBER) {
            /* reading R36: on amber a vehicle goes on iff it could not stop before the line at the
             * comfortable deceleration b: v^2 > 2 b (C - x) */
            float rem = Cf - x;
            float vv = v * v;
            float need = S->two_b * rem;
            may_cross = vv > need;
        }
    } else if (!last && ctrl == CTRL_STOP) {
        /* reading R34 ("allows just one vehicle at a time into the intersection and
         * waits until the car has reached the next edge"): the line is a standing obstacle until
         * the vehicle has come to a halt at it (within stop_dist of the line at no more than
         * stop_speed) AND the node is not held by a vehicle that crossed it earlier */
        float rem = Cf - x;
        if (rem <= p->stop_dist && v <= p->stop_speed) made_stop = 1;
        may_cross = made_stop && S->node_free_from[h] <= k;
    }
    S->stop_t[i] = made_stop;
    const int32_t c = cell_of(S, i);
    cnt->updates++;

    /* 2b own leader: nearest occupied cell with c < cL <= min(C-1, c+H) */
    int has_lead = 0, lead_on_edge = 0;
    float s_lead = 0.0f, dv_lead = 0.0f;
    {
        int32_t lim = c + H < C - 1 ? c + H : C - 1;
        int32_t j = S->ahead[i];
        if (j != NONE && cell_of(S, (uint32_t)j) <= lim) {
            int32_t cL = cell_of(S, (uint32_t)j);
            has_lead = 1; lead_on_edge = 1;
            s_lead = (float)cL - S->t_len[S->veh_type[j]];   /* E3 same edge: the LEADER's length */
            s_lead = s_lead - x;
            dv_lead = v - orc_speed_decode(orc_speed_code(S->v[j]));
            cnt->own_cells += (uint64_t)(cL - c); cnt->own_chunks16 += (uint64_t)(cL - c + 15) / 16;
        } else {
            cnt->own_cells += (uint64_t)(lim - c); cnt->own_chunks16 += (uint64_t)(lim - c + 15) / 16;
            int32_t Hp = H - (C - 1 - c);
            if (!last && may_cross && Hp > 0) {
                int32_t C2 = (int32_t)S->edge_len[e2];
                int32_t lim2 = Hp - 1 < C2 - 1 ? Hp - 1 : C2 - 1;
                int32_t j2 = S->lane_tail[S->lane_base[e2] + l2];
                if (j2 != NONE && cell_of(S, (uint32_t)j2) <= lim2) {
                    int32_t cL2 = cell_of(S, (uint32_t)j2);
                    has_lead = 1;
                    s_lead = Cf - x;            /* E3 across the node */
                    s_lead = s_lead + (float)cL2;
                    s_lead = s_lead - S->t_len[S->veh_type[j2]];
                    dv_lead = v - orc_speed_decode(orc_speed_code(S->v[j2]));
                    cnt->next_cells += (uint64_t)(cL2 + 1); cnt->next_chunks16 += (uint64_t)(cL2 + 1 + 15) / 16;
                } else {
                    cnt->next_cells += (uint64_t)(lim2 + 1); cnt->next_chunks16 += (uint64_t)(lim2 + 1 + 15) / 16;
                }
            }
        }
    }

    /* 2d lane change (readings R10-R14) */
    int accepted = 0, has_Lt = 0;
    float s_Lt = 0.0f, at_c = 0.0f;
    uint32_t lt = l;
    if (p->lc_period != 0 && lanes_e >= 2) {
        int dir = (k & 1) ? -1 : +1;
        int32_t lti = (int32_t)l + dir;
        float n = a_i * p->dt;                  /* E5 cannot cross this step */
        n = v + n;
        n = n * p->dt;
        n = x + n;
        if (lti >= 0 && lti < (int32_t)lanes_e && x >= (float)p->entry_zone_cells && n < Cf &&
            ((k >> 1) + i) % p->lc_period == 0) {
            lt = (uint32_t)lti;
            cnt->lc_evals++;
            int32_t jl, jf;
            lane_neighbours(S, S->lane_base[e] + lt, c, &jl, &jf);
            int32_t lim = c + H < C - 1 ? c + H : C - 1;
            int32_t lo = c - Hb > 0 ? c - Hb : 0;
            int has_F = 0;
            int32_t cLt = 0, cF = 0;
            float vLt = 0.0f, vF = 0.0f, s_lag = 0.0f, len_Lt = 0.0f;
            uint32_t tyF = 0;
            if (jl != NONE && cell_of(S, (uint32_t)jl) <= lim) {
                has_Lt = 1; cLt = cell_of(S, (uint32_t)jl);
                vLt = orc_speed_decode(orc_speed_code(S->v[jl]));
                len_Lt = S->t_len[S->veh_type[jl]];
                s_Lt = (float)cLt - len_Lt;
                s_Lt = s_Lt - x;
                cnt->lc_cells += (uint64_t)(cLt - c + 1); cnt->lc_chunks16 += (uint64_t)(cLt - c + 1 + 15) / 16;
            } else { cnt->lc_cells += (uint64_t)(lim - c + 1); cnt->lc_chunks16 += (uint64_t)(lim - c + 1 + 15) / 16; }
            if (jf != NONE && cell_of(S, (uint32_t)jf) >= lo) {
                has_F = 1; cF = cell_of(S, (uint32_t)jf);
                tyF = S->veh_type[jf];
                vF = orc_speed_decode(orc_speed_code(S->v[jf]));
                s_lag = x - len;                /* E3 lag */
                s_lag = s_lag - (float)(cF + 1);
                cnt->lc_cells += (uint64_t)(c - cF); cnt->lc_chunks16 += (uint64_t)(c - cF + 15) / 16;
            } else { cnt->lc_cells += (uint64_t)(c - lo); cnt->lc_chunks16 += (uint64_t)(c - lo + 15) / 16; }

            int ok = 1;
            float aF_new = 0.0f;
            /* what the changer knows of the lag vehicle's desired speed: the edge limit, capped by its type */
            float v0F = fminf(S->edge_vlim[e], S->t_vmax[tyF]);
            if (has_Lt && !(s_Lt >= p->s0)) ok = 0;                         /* G1 */
            if (ok && has_F) {                                              /* G2 */
                float m = 0.5f * S->t_a[tyF];   /* E4, with the lag vehicle's acceleration ability */
                m = m * p->dt;
                m = (vF + 0.125f) + m;
                m = m * p->dt;
                if (!(s_lag >= p->s0 && s_lag >= m)) ok = 0;
            }
            if (ok && has_F) {                                              /* G3 */
                aF_new = idm(S, tyF, vF, v0F, 1, s_lag, vF - v);
                if (!(aF_new >= -p->b_safe)) ok = 0;
            }
            if (ok) {                                                       /* G4 */
                float rem = Cf - x;
                int mandatory = !last && l >= lanes_e2 && lt < l && rem <= S->mand_dist[i];
                at_c = idm(S, ty, v, v0, has_Lt, s_Lt, v - vLt);
                if (mandatory) { accepted = 1; cnt->lc_mandatory++; }
                else if (!last && lt >= lanes_e2 && rem <= S->mand_dist[i]) accepted = 0;
                else {
                    float a_c = lead_on_edge ? idm(S, ty, v, v0, 1, s_lead, dv_lead)
                                             : idm(S, ty, v, v0, 0, 0.0f, 0.0f);
                    float inc = at_c - a_c;
                    if (has_F) {
                        float sF = (float)cLt - len_Lt;
                        sF = sF - (float)(cF + 1);
                        float a_F = idm(S, tyF, vF, v0F, has_Lt, sF, vF - vLt);
                        float d2 = aF_new - a_F;
                        d2 = p->politeness * d2;
                        inc = inc + d2;
                    }
                    accepted = inc > p->lc_threshold;
                }
            }
            if (accepted) cnt->lc_accepts++;
        }
    }

    /* 2e acceleration and integration (E2, reading R3) */
    float acc = idm(S, ty, v, v0, has_lead, s_lead, dv_lead);
    if (!may_cross) {                            /* 2c stop line as a standing obstacle (R17) */
        float s_stop = Cf - x;
        acc = fminf(acc, idm(S, ty, v, v0, 1, s_stop, v));
    }
    float cap = INFINITY;
    if (has_lead) cap = fmaxf(s_lead, 0.0f);
    if (accepted && has_Lt) { acc = fminf(acc, at_c); cap = fminf(cap, fmaxf(s_Lt, 0.0f)); }
    float vt = acc * p->dt;
    vt = v + vt;
    vt = fmaxf(vt, 0.0f);
    vt = fminf(vt, v0);
    float dx = v + vt;
    dx = 0.5f * dx;
    dx = dx * p->dt;
    if (dx > cap) { dx = cap; vt = 0.0f; cnt->cap_bound++; }
    float xt = x + dx;

    /* section 6.3.4: "since it has the position, speed, acceleration of each
     * vehicle at every given time".  Reading R30: every step each ACTIVE vehicle adds rate * dt
     * (the paper updates "every second"; with dt = 0.5 s this is the same integral on the
     * simulation's own grid), with the speed v of state k and the acceleration of this step as
     * integrated by E2, ar = (vt - v) * (1/dt), 1/dt rounded once.  A later hold at the line or
     * a lost claim (which zero the speed) is not fed back into this step's rate. */
    if (p->emissions) {
        float inv_dt = 1.0f / p->dt;
        float ar = vt - v;
        ar = ar * inv_dt;
        float e = orc_co_rate(v);
        e = e * p->dt;
        S->co_g[i] = S->co_g[i] + e;
        float f = orc_fuel_rate(v, ar);
        f = f * p->dt;
        S->fuel_ml[i] = S->fuel_ml[i] + f;
    }

    /* 2f */
    uint8_t act = ACT_STAY;
    if (xt >= Cf) {
        if (last) act = ACT_ARRIVE;
        else if (may_cross) {
            act = ACT_CROSS;                    /* its claims are posted by post_claims() */
        } else { xt = Cf - 0.0625f; vt = 0.0f; cnt->held_red++; }
    }
    S->xt[i] = xt; S->vt[i] = vt; S->act[i] = act;
    S->ln[i] = (uint8_t)(accepted ? lt : l);
    S->e2[i] = e2; S->l2[i] = (uint8_t)l2;
}

/* SURVEY.md 8(c) step 2f, second half: a CROSS intent claims its target lane and, at a PRIORITY
 * node, the node (claim = minimum id).  Kept apart from vehicle_intent() so that the intents,
 * which read state k only and write only the vehicle's own intent (I8), may be evaluated by
 * several host threads (orc_set_threads); the claims are posted by one thread. */
static void post_claims(orc_sim *S, uint32_t i) {
    if (S->act[i] != ACT_CROSS) return;
    uint32_t h = S->edge_to[S->edge[i]];
    claim_lane(S, S->lane_base[S->e2[i]] + S->l2[i], i);
    if (S->node_ctrl[h] == CTRL_PRIORITY || S->node_ctrl[h] == CTRL_STOP) claim_node(S, h, i);
}

/* departure intent of queue q. */
static void departure_intent(orc_sim *S, uint32_t q) {
    S->dep_cand[q] = NO_CLAIM;
    if (S->queue_head[q] == S->queue_off[q + 1]) return;
    uint32_t i = S->queue_veh[S->queue_head[q]];
    if (S->dep_step[i] > S->k) return;
    uint32_t e = S->queue_edge[q];
    uint64_t g = S->lane_base[e];               /* lane 0 = kerb side (reading R18) */
    int32_t j = S->lane_tail[g];
    if (j != NONE && cell_of(S, (uint32_t)j) < (int32_t)S->p.insert_clear_cells) return;
    S->dep_cand[q] = i;
    claim_lane(S, g, i);
}

/* ---------------------------------------------------------------- lane lists */

static void list_unlink(orc_sim *S, uint32_t i, uint64_t g) {
    int32_t a = S->ahead[i], b = S->behind[i];
    if (a != NONE) S->behind[a] = b; else S->lane_head[g] = b;
    if (b != NONE) S->ahead[b] = a; else S->lane_tail[g] = a;
    S->ahead[i] = NONE; S->behind[i] = NONE;
}

/* Insert i into lane g at the place its (already committed) position gives it. */
static void list_insert(orc_sim *S, uint32_t i, uint64_t g) {
    int32_t ci = cell_of(S, i);
    int32_t j = S->lane_tail[g], prev = NONE;
    while (j != NONE && cell_of(S, (uint32_t)j) < ci) { prev = j; j = S->ahead[j]; }
    S->ahead[i] = j; S->behind[i] = prev;
    if (j != NONE) S->behind[j] = (int32_t)i; else S->lane_head[g] = (int32_t)i;
    if (prev != NONE) S->ahead[prev] = (int32_t)i; else S->lane_tail[g] = (int32_t)i;
}

static void active_add(orc_sim *S, uint32_t i) {
    S->active_pos[i] = S->n_active_list; S->active[S->n_active_list++] = i;
}
static void active_remove(orc_sim *S, uint32_t i) {
    uint32_t pos = S->active_pos[i], lastv = S->active[--S->n_active_list];
    S->active[pos] = lastv; S->active_pos[lastv] = pos;
}

/* ---------------------------------------------------------------- invariants (I1-I7, P4) */

/* O(V) search over raw (edge, lane, x): rear-most ACTIVE vehicle with cell >= c_from and
 * front-most with cell < c_from on lane (e,l).  Independent of the lane lists. */
static void brute_neighbours(const orc_sim *S, uint32_t e, uint32_t l, int32_t c_from,
                             int32_t *lead, int32_t *lag) {
    *lead = NONE; *lag = NONE;
    for (uint32_t j = 0; j < S->V; j++) {
        if (S->status[j] != ST_ACTIVE || S->edge[j] != e || S->lane[j] != l) continue;
        int32_t cj = cell_of(S, j);
        if (cj >= c_from) { if (*lead == NONE || cj < cell_of(S, (uint32_t)*lead)) *lead = (int32_t)j; }
        else { if (*lag == NONE || cj > cell_of(S, (uint32_t)*lag)) *lag = (int32_t)j; }
    }
}

static int check_brute(const orc_sim *S) {
    for (uint32_t n = 0; n < S->n_active_list; n++) {
        uint32_t i = S->active[n];
        uint32_t e = S->edge[i], l = S->lane[i];
        int32_t c = cell_of(S, i), bl, bf, ll, lf;
        brute_neighbours(S, e, l, c + 1, &bl, &bf);
        if (bl != S->ahead[i]) { FAIL("P4: step %llu veh %u own leader list %d brute %d", (unsigned long long)S->k, i, S->ahead[i], bl); return -1; }
        if (bf != (int32_t)i) { FAIL("P4: step %llu veh %u not rear neighbour of itself", (unsigned long long)S->k, i); return -1; }
        for (uint32_t lt = 0; lt < S->edge_lanes[e]; lt++) {
            if (lt == l) continue;
            brute_neighbours(S, e, lt, c, &bl, &bf);
            lane_neighbours(S, S->lane_base[e] + lt, c, &ll, &lf);
            if (bl != ll || bf != lf) { FAIL("P4: step %llu veh %u lane %u neighbours", (unsigned long long)S->k, i, lt); return -1; }
        }
        uint64_t rpos = S->route_off[i] + S->r[i];
        if (rpos + 1 < S->route_off[i + 1]) {
            uint32_t e2 = S->route_edges[rpos + 1];
            for (uint32_t q = 0; q < S->edge_lanes[e2]; q++) {
                brute_neighbours(S, e2, q, 0, &bl, &bf);
                if (bl != S->lane_tail[S->lane_base[e2] + q]) { FAIL("P4: step %llu veh %u next-edge tail", (unsigned long long)S->k, i); return -1; }
            }
        }
    }
    return 0;
}

static int check_invariants(const orc_sim *S) {
    unsigned long long k = (unsigned long long)S->k;
    /* I1 conservation */
    if ((uint64_t)S->n_pending + S->n_active + S->n_arrived != S->V || S->n_active != S->n_active_list) {
        FAIL("I1: step %llu counts %u+%u+%u != %u", k, S->n_pending, S->n_active, S->n_arrived, S->V); return -1;
    }
    uint64_t in = 0, out = 0;
    for (uint32_t e = 0; e < S->E; e++) { in += S->entered[e]; out += S->exited[e]; }
    if (in - out != S->n_active) { FAIL("I1: step %llu entered-exited %llu != active %u", k, (unsigned long long)(in - out), S->n_active); return -1; }
    /* lists: I2 exclusivity + I3 order (cells strictly increasing tail -> head) */
    uint64_t listed = 0;
    for (uint32_t e = 0; e < S->E; e++)
        for (uint32_t l = 0; l < S->edge_lanes[e]; l++) {
            uint64_t g = S->lane_base[e] + l;
            int32_t prev = NONE;
            for (int32_t j = S->lane_tail[g]; j != NONE; j = S->ahead[j]) {
                if (S->status[j] != ST_ACTIVE || S->edge[j] != e || S->lane[j] != l) { FAIL("list: step %llu veh %d in wrong list", k, j); return -1; }
                if (S->behind[j] != prev) { FAIL("list: step %llu veh %d back link", k, j); return -1; }
                if (prev != NONE && cell_of(S, (uint32_t)prev) >= cell_of(S, (uint32_t)j)) { FAIL("I2/I3: step %llu veh %d and %d share or swap cells on edge %u lane %u", k, prev, j, e, l); return -1; }
                prev = j; listed++;
            }
            if (S->lane_head[g] != prev) { FAIL("list: step %llu head of edge %u lane %u", k, e, l); return -1; }
        }
    if (listed != S->n_active) { FAIL("list: step %llu %llu listed, %u active", k, (unsigned long long)listed, S->n_active); return -1; }
    /* I4 speed range, I5 position range, route consistency */
    for (uint32_t n = 0; n < S->n_active_list; n++) {
        uint32_t i = S->active[n], e = S->edge[i];
        float v0 = fminf(S->v0_mult[i] * S->edge_vlim[e], S->t_vmax[S->veh_type[i]]);
        if (!(S->v[i] >= 0.0f && S->v[i] <= v0)) { FAIL("I4: step %llu veh %u v=%g v0=%g", k, i, S->v[i], v0); return -1; }
        if (!(S->x[i] >= 0.0f && S->x[i] < (float)S->edge_len[e])) { FAIL("I5: step %llu veh %u x=%g C=%u", k, i, S->x[i], S->edge_len[e]); return -1; }
        if (S->route_edges[S->route_off[i] + S->r[i]] != e) { FAIL("I1: step %llu veh %u off route", k, i); return -1; }
    }
    return 0;
}

/* ---------------------------------------------------------------- one step: resolve + commit */

static uint64_t vehicle_hash(uint32_t id, uint32_t edge, uint32_t lane, float x, float v) {
    uint64_t g = orc_mix64((uint64_t)id);
    g = orc_mix64(g ^ (((uint64_t)edge << 8) | (uint64_t)lane));
    g = orc_mix64(g ^ (((uint64_t)fbits(x) << 32) | (uint64_t)fbits(v)));
    return g;
}

static uint64_t step_digest(const orc_sim *S) {
    uint64_t d = 0;
    for (uint32_t n = 0; n < S->n_active_list; n++) {
        uint32_t i = S->active[n];
        d += vehicle_hash(i, S->edge[i], S->lane[i], S->x[i], S->v[i]);
    }
    uint64_t g = orc_mix64((uint64_t)S->n_pending);
    g = orc_mix64(g ^ (uint64_t)S->n_active);
    g = orc_mix64(g ^ (uint64_t)S->n_arrived);
    g = orc_mix64(g ^ S->sum_arrive_step);
    return d + g;
}

static void shuffle_active(orc_sim *S, uint64_t seed) {
    uint64_t z = seed;
    for (uint32_t n = S->n_active_list; n > 1; n--) {
        z = orc_mix64(z);
        uint32_t m = (uint32_t)(z % n);
        uint32_t a = S->active[n - 1], b = S->active[m];
        S->active[n - 1] = b; S->active[m] = a;
        S->active_pos[b] = n - 1; S->active_pos[a] = m;
    }
}

/* The intent loop of step 2 on S->threads host threads (OpenMP).  Licensed by the synchronous
 * update: vehicle_intent() reads state k and writes only vehicle i's own intent, so the loop's
 * iterations are independent (the same property as I8).  The arithmetic is vehicle_intent()'s,
 * untouched; work counters are kept per thread and added up.  Used only to get through the
 * multi-hour whole-run traces of tests/golden/make_golden.py; the default is one thread. */
static void intents_threaded(orc_sim *S) {
    enum { MAXT = 64 };
    static orc_counters zero;
    orc_counters part[MAXT];
    int T = S->threads > MAXT ? MAXT : S->threads;
    for (int t = 0; t < T; t++) part[t] = zero;
    long n_act = (long)S->n_active_list;
#ifdef _OPENMP
#pragma omp parallel num_threads(T)
    {
        orc_counters *cnt = &part[omp_get_thread_num()];
#pragma omp for schedule(static)
        for (long n = 0; n < n_act; n++) vehicle_intent(S, S->active[n], cnt);
    }
#else
    for (long n = 0; n < n_act; n++) vehicle_intent(S, S->active[n], &part[0]);
#endif
    uint64_t *dst = (uint64_t *)&S->cnt;
    for (int t = 0; t < T; t++) {
        const uint64_t *src = (const uint64_t *)&part[t];
        for (size_t f = 0; f < sizeof(orc_counters) / 8; f++) dst[f] += src[f];
    }
}

void orc_set_threads(orc_sim *S, int n) { S->threads = n < 1 ? 1 : n; }

static int one_step(orc_sim *S, int check, uint64_t order_seed) {
    const uint64_t k = S->k;
    const uint32_t k1 = (uint32_t)(k + 1);
    if (order_seed) shuffle_active(S, order_seed + k);
    if (check >= 2 && check_brute(S)) return -1;

    /* steps 1-3: intents from state k */
    S->n_touched_lanes = 0; S->n_touched_nodes = 0;
    if (S->threads > 1) intents_threaded(S);
    else for (uint32_t n = 0; n < S->n_active_list; n++) vehicle_intent(S, S->active[n], &S->cnt);
    for (uint32_t n = 0; n < S->n_active_list; n++) post_claims(S, S->active[n]);
    for (uint32_t q = 0; q < S->n_queues; q++) departure_intent(S, q);

    /* step 4: resolve + commit.  Only own intent and the claim words are read here. */
    S->n_relink = 0; S->n_entry = 0; S->n_cross_node = 0;
    uint32_t n_snapshot = S->n_active_list;
    for (uint32_t n = n_snapshot; n-- > 0;) {       /* backwards: removal swaps in a visited entry */
        uint32_t i = S->active[n];
        uint32_t e = S->edge[i], l = S->lane[i];
        uint64_t g = S->lane_base[e] + l;
        float Cf = (float)S->edge_len[e];
        float x_old = S->x[i], v_old = S->v[i];
        /* reading R34: a vehicle that holds the STOP node at the tail of its edge lets go once its
         * rear bumper is past it (always the case by the time it leaves the edge: len < 16 <= C);
         * the node is free again from the next step on */
        if (S->owns_node[i] && S->xt[i] >= S->t_len[S->veh_type[i]]) {
            S->node_free_from[S->edge_from[e]] = k1;
            S->owns_node[i] = 0;
        }
        S->made_stop[i] = S->stop_t[i];
        if (S->act[i] == ACT_CROSS) {
            uint32_t e2 = S->e2[i], l2 = S->l2[i], h = S->edge_to[e];
            uint64_t g2 = S->lane_base[e2] + l2;
            uint32_t ctrl = S->node_ctrl[h];
            int win = S->lane_claim[g2] == i &&
                      ((ctrl != CTRL_PRIORITY && ctrl != CTRL_STOP) || S->node_claim[h] == i);
            if (win) {
                if (check && (ctrl == CTRL_SIGNAL || ctrl == CTRL_SIGNAL_NM) &&
                    orc_signal_phase(S->sig_green[h], S->p.amber_steps, S->sig_allred[h], S->sig_offset[h], S->node_n_in[h],
                                     ctrl == CTRL_SIGNAL_NM ? S->node_n_out[h] : 0, S->edge_in_rank[e], S->edge_out_rank[e2], k) == SIG_RED) {
                    FAIL("I7: step %llu veh %u crossed on red", (unsigned long long)k, i); return -1;
                }
                if (check && ctrl == CTRL_STOP && !(S->node_free_from[h] <= k)) {
                    FAIL("I7: step %llu veh %u crossed a STOP node that was held", (unsigned long long)k, i); return -1;
                }
                if (ctrl == CTRL_STOP) {             /* holds the node until it has cleared it */
                    S->node_free_from[h] = UINT32_MAX;
                    S->owns_node[i] = 1;
                }
                S->made_stop[i] = 0;
                float xn = S->xt[i] - Cf;
                xn = fminf(xn, (float)S->edge_len[e2] - 0.0625f);
                float v0n = S->v0_mult[i] * S->edge_vlim[e2];
                v0n = fminf(v0n, S->t_vmax[S->veh_type[i]]);
                list_unlink(S, i, g);
                S->x[i] = xn; S->v[i] = fminf(S->vt[i], v0n);      /* reading R9 */
                S->edge[i] = e2; S->lane[i] = (uint8_t)l2; S->r[i]++;
                S->entered[e2]++; S->exited[e]++;
                S->exit_steps_sum[e] += (uint64_t)(k1 - S->enter_step[i]);
                S->enter_step[i] = k1;
                S->relink[S->n_relink++] = i;
                S->entry_lane[S->n_entry++] = g2;
                if (ctrl == CTRL_PRIORITY || ctrl == CTRL_STOP) S->cross_node[S->n_cross_node++] = h;
                S->cnt.crossings++;
            } else {                                               /* reading R15: held at the line */
                S->x[i] = Cf - 0.0625f; S->v[i] = 0.0f;
                S->cnt.cross_lost++;
            }
        } else if (S->act[i] == ACT_ARRIVE) {
            list_unlink(S, i, g);
            S->status[i] = ST_ARRIVED; S->arrive_step[i] = k1;
            S->x[i] = Cf; S->v[i] = S->vt[i];
            S->exited[e]++;
            S->exit_steps_sum[e] += (uint64_t)(k1 - S->enter_step[i]);
            active_remove(S, i);
            S->n_active--; S->n_arrived++; S->sum_arrive_step += k1;
            S->cnt.arrivals++;
        } else {
            S->x[i] = S->xt[i]; S->v[i] = S->vt[i];
            if (S->ln[i] != l) {
                list_unlink(S, i, g);
                S->lane[i] = S->ln[i];
                S->relink[S->n_relink++] = i;
            }
        }
        if (check && S->status[i] == ST_ACTIVE && S->edge[i] == e) {  /* I5 advance bound */
            double bound = ((double)v_old + 0.5 * S->t_a[S->veh_type[i]] * S->p.dt) * S->p.dt + 1e-3;
            if ((double)S->x[i] - (double)x_old > bound) { FAIL("I5: step %llu veh %u advanced %g > %g", (unsigned long long)k, i, S->x[i] - x_old, bound); return -1; }
        }
    }
    for (uint32_t q = 0; q < S->n_queues; q++) {
        uint32_t i = S->dep_cand[q];
        if (i == NO_CLAIM) continue;
        uint32_t e = S->queue_edge[q];
        if (S->lane_claim[S->lane_base[e]] != i) continue;
        S->status[i] = ST_ACTIVE; S->x[i] = 0.0f; S->v[i] = 0.0f; S->lane[i] = 0; S->r[i] = 0;
        S->edge[i] = e; S->insert_step[i] = k1; S->enter_step[i] = k1;
        S->entered[e]++; S->queue_head[q]++;
        S->n_pending--; S->n_active++;
        active_add(S, i);
        S->relink[S->n_relink++] = i;
        S->entry_lane[S->n_entry++] = S->lane_base[e];
        S->cnt.departures++;
    }
    if (check) {   /* I7: at most one entry per lane and one crossing per PRIORITY node per step */
        for (uint32_t a = 0; a < S->n_entry; a++)
            for (uint32_t b = a + 1; b < S->n_entry; b++)
                if (S->entry_lane[a] == S->entry_lane[b]) { FAIL("I7: step %llu two entries into one lane", (unsigned long long)k); return -1; }
        for (uint32_t a = 0; a < S->n_cross_node; a++)
            for (uint32_t b = a + 1; b < S->n_cross_node; b++)
                if (S->cross_node[a] == S->cross_node[b]) { FAIL("I7: step %llu two crossings of PRIORITY node %u", (unsigned long long)k, S->cross_node[a]); return -1; }
    }
    /* every position is committed: put movers into their new lists */
    for (uint32_t n = 0; n < S->n_relink; n++) {
        uint32_t i = S->relink[n];
        list_insert(S, i, S->lane_base[S->edge[i]] + S->lane[i]);
    }
    for (uint64_t n = 0; n < S->n_touched_lanes; n++) S->lane_claim[S->touched_lanes[n]] = NO_CLAIM;
    for (uint32_t n = 0; n < S->n_touched_nodes; n++) S->node_claim[S->touched_nodes[n]] = NO_CLAIM;
    if (S->n_active > S->cnt.peak_active) S->cnt.peak_active = S->n_active;

    S->k = k + 1;
    /* step 5: sampling ("we sample every minute the utilization and per edge speed") */
    if (S->p.sample_period_steps && S->k % S->p.sample_period_steps == 0) {
        for (uint32_t n = 0; n < S->n_active_list; n++) {
            uint32_t i = S->active[n];
            S->sample_count_sum[S->edge[i]]++;
            S->sample_speedcode_sum[S->edge[i]] += (uint64_t)(orc_speed_code(S->v[i]) - 1);
        }
        S->n_samples++;
    }
    if (check && check_invariants(S)) return -1;
    return 0;
}

int orc_step(orc_sim *S, uint32_t n, uint64_t *digests, int check, uint64_t order_seed) {
    for (uint32_t s = 0; s < n; s++) {
        if (one_step(S, check, order_seed)) return -1;
        if (digests) digests[s] = step_digest(S);
    }
    return 0;
}

/* ---------------------------------------------------------------- read-back */

void orc_read_state(const orc_sim *S, uint8_t *status, uint32_t *edge, uint8_t *lane,
                    uint32_t *cell, float *x, float *v, uint32_t *route_idx,
                    uint32_t *insert_step, uint32_t *arrive_step,
                    uint64_t *step, uint32_t *n_pending, uint32_t *n_active,
                    uint32_t *n_arrived) {
    for (uint32_t i = 0; i < S->V; i++) {
        if (status) status[i] = S->status[i];
        if (edge) edge[i] = S->edge[i];
        if (lane) lane[i] = S->lane[i];
        if (cell) cell[i] = (uint32_t)floorf(S->x[i]);
        if (x) x[i] = S->x[i];
        if (v) v[i] = S->v[i];
        if (route_idx) route_idx[i] = S->r[i];
        if (insert_step) insert_step[i] = S->insert_step[i];
        if (arrive_step) arrive_step[i] = S->arrive_step[i];
    }
    if (step) *step = S->k;
    if (n_pending) *n_pending = S->n_pending;
    if (n_active) *n_active = S->n_active;
    if (n_arrived) *n_arrived = S->n_arrived;
}

void orc_read_edge_stats(orc_sim *S, uint32_t *entered, uint32_t *exited,
                         uint64_t *exit_steps_sum, uint32_t *sample_count_sum,
                         uint64_t *sample_speedcode_sum, uint32_t *n_samples, int reset) {
    size_t E = S->E;
    if (entered) memcpy(entered, S->entered, E * 4);
    if (exited) memcpy(exited, S->exited, E * 4);
    if (exit_steps_sum) memcpy(exit_steps_sum, S->exit_steps_sum, E * 8);
    if (sample_count_sum) memcpy(sample_count_sum, S->sample_count_sum, E * 4);
    if (sample_speedcode_sum) memcpy(sample_speedcode_sum, S->sample_speedcode_sum, E * 8);
    if (n_samples) *n_samples = S->n_samples;
    if (reset) {
        memset(S->entered, 0, E * 4); memset(S->exited, 0, E * 4);
        memset(S->exit_steps_sum, 0, E * 8); memset(S->sample_count_sum, 0, E * 4);
        memset(S->sample_speedcode_sum, 0, E * 8); S->n_samples = 0;
    }
}

void orc_read_emissions(const orc_sim *S, float *co_g, float *fuel_ml) {
    if (co_g) memcpy(co_g, S->co_g, (size_t)S->V * 4);
    if (fuel_ml) memcpy(fuel_ml, S->fuel_ml, (size_t)S->V * 4);
}

void orc_get_counters(const orc_sim *S, orc_counters *out) { *out = S->cnt; }
