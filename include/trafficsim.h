/*
 * trafficsim.h -- C ABI of the B200-native traffic microsimulation (libts.so).
 *
 * What it computes: the time-stepped, per-vehicle traffic simulation of arxiv 1807.01148,
 * section 6.3.2 "Per-vehicle and traffic control simulation" (Intelligent
 * Driver Model car following Eq. 7, mandatory/discretionary lane changes, gap acceptance,
 * stop and traffic-light control) on the "traffic atlas" of section 6.3.3 (PAPER.md:404-406:
 * "we represent a road as a set of contiguous bytes in memory, in order to find the leading
 * car of a given vehicle, we check the following bytes"), along per-vehicle paths
 * (PAPER.md:370, :382-384), with the outputs of section 6.4.
 * The exact rule set (one synchronous step k -> k+1, readings R1-R22 where the paper is
 * silent) is written out in DESIGN.md sections 2-3.
 *
 * Conventions
 *  - No global state, no exceptions, no allocation on the device by the library: the caller
 *    owns ONE device workspace (size from ts_query_workspace) and a CUDA stream.
 *  - Every pointer inside ts_network / ts_routes / ts_departures is a HOST pointer owned by
 *    the caller; ts_create copies what it needs and keeps no pointer afterwards.
 *  - Output pointers (ts_state_out, ts_edge_stats_out, digests) are HOST pointers unless
 *    ts_device.out_on_device != 0, in which case they are DEVICE pointers.
 *  - All calls on one ts_sim must come from one thread at a time.  Work is enqueued on
 *    ts_device.cuda_stream; ts_step is asynchronous, the ts_read_* calls synchronise.
 *  - Return value: TS_OK (0) or a negative ts_status; ts_last_error() gives the message.
 *  - fp32 state is reproducible bit for bit: kernels are built with -fmad=false and IEEE
 *    division; arbitration is by lowest vehicle id with integer atomics only.
 *  - There is no CPU fallback: without a CUDA device every call but ts_query_workspace,
 *    ts_last_error and ts_version fails with TS_ECUDA.
 */
#ifndef TRAFFICSIM_H
#define TRAFFICSIM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum ts_status {
    TS_OK = 0,
    TS_EINVAL = -1,     /* bad sizes, non-contiguous route, lanes not in 1..8, edge shorter than
                           16 or longer than 65535 cells, entry zone too short for the fastest
                           vehicle, lookahead not a multiple of 16, ... */
    TS_ENOMEM = -2,     /* workspace too small */
    TS_ECUDA = -3,      /* CUDA runtime error (or no device) */
    TS_EINVARIANT = -4  /* device-side sticky flag: two vehicles scattered to one cell; a position or
                           speed that is NaN, negative or infinite; two vehicles of one lane closer
                           than the 4-cell granule of the atlas's code plane (cannot happen under the
                           rule set with vehicles of 4 m or more: it means the state is corrupt) */
} ts_status;

/* Node control types ("stop and traffic light signals"). */
/* Controls ("Our system implements stop and traffic light signals"):
 *  FREE       no control.
 *  PRIORITY   at most one vehicle crosses the node per step, lowest id first (reading R15).
 *  SIGNAL     fixed-time light, one phase per inbound edge in round robin (reading R16).
 *  STOP       "allows just one vehicle at a time into the intersection and waits until the car has
 *             reached the next edge": every vehicle first comes to a halt at the line (ts_params
 *             stop_dist / stop_speed), then crosses when the node is free, lowest id first, and
 *             holds the node until its rear bumper is past it (reading R34).
 *  SIGNAL_NM  "given an intersection with n inbound edges and m outbound, our system creates the
 *             geometric combination nm of necessary traffic phasing ... round robin": one phase per
 *             movement (inbound i, outbound j), number i*m + j, ranks by edge index (reading R35).
 * Every signal phase is green, then ts_params.amber_steps of amber (R36), then all-red. */
enum { TS_CTRL_FREE = 0, TS_CTRL_PRIORITY = 1, TS_CTRL_SIGNAL = 2, TS_CTRL_STOP = 3, TS_CTRL_SIGNAL_NM = 4 };
/* Vehicle status. */
enum { TS_PENDING = 0, TS_ACTIVE = 1, TS_ARRIVED = 2 };

/* The road network (nodes, directional edges, per-edge speed and lanes). */
typedef struct ts_network {
    uint32_t n_nodes, n_edges;
    const uint32_t *edge_from;        /* [E] tail node */
    const uint32_t *edge_to;          /* [E] head node */
    const uint32_t *edge_len_m;       /* [E] length in cells = metres, 16..65535 */
    const uint8_t *edge_lanes;        /* [E] 1..8, lane 0 = kerb side */
    const float *edge_vlim;           /* [E] speed limit m/s, > 0 */
    const uint8_t *node_ctrl;         /* [N] TS_CTRL_* of the node at the head of an edge */
    const uint32_t *sig_green_steps;  /* [N] read where ctrl == SIGNAL; >= 1; green+allred <= 65535 */
    const uint32_t *sig_allred_steps; /* [N] */
    const uint32_t *sig_offset_steps; /* [N] < 2^31 */
} ts_network;

/* Per-vehicle paths.  Vehicle id = index.  Each route has >= 1 edge and
 * head(route[j]) == tail(route[j+1]). */
typedef struct ts_routes {
    uint32_t n_vehicles;
    const uint64_t *route_off;        /* [V+1] */
    const uint32_t *route_edges;      /* [route_off[V]] */
} ts_routes;

/* Departure times and per-vehicle procedural variables. */
typedef struct ts_departures {
    const float *depart_time_s;       /* [V] >= 0; departs at step ceil(t/dt) or later */
    const float *v0_mult;             /* [V] desired speed = v0_mult * edge limit; NULL => 1 */
    const float *mand_dist_m;         /* [V] distance to the exit at which a wrong-lane vehicle
                                         turns mandatory; NULL => default */
    const uint8_t *veh_type;          /* [V] vehicle type < max(1, ts_params.n_types) (PAPER.md:433:
                                         "a second type of vehicle to represent trucks"); NULL => 0 */
} ts_departures;

/* Model parameters.  Defaults in DESIGN.md section 3 (BASELINE.json configs 1-2). */
typedef struct ts_params {
    float dt;                 /* s, PAPER.md:390 (0.5) */
    float a, b, T, s0;        /* IDM, Eq. 7 */
    float veh_len;            /* m, >= 2 */
    float b_safe;             /* gap acceptance: max braking imposed on the lag vehicle */
    float politeness;         /* MOBIL p */
    float lc_threshold;       /* MOBIL incentive threshold m/s^2 */
    float mand_dist_default;  /* m */
    uint32_t lookahead_cells; /* H: multiple of 16, 16..4096 */
    uint32_t lookback_cells;  /* Hb */
    uint32_t lc_period;       /* lane change evaluated when ((k>>1)+id) % lc_period == 0; 0 = never */
    uint32_t entry_zone_cells;   /* no lane change in the first cells of an edge */
    uint32_t insert_clear_cells; /* 1..16: cells of lane 0 that must be empty to insert */
    uint32_t sample_period_steps;/* PAPER.md:437 (120 = one minute); 0 = never */
    uint32_t emissions;          /* non-zero: keep per-vehicle CO (Eq. 8) and fuel
                                    (Eq. 9) totals; costs 8 bytes per vehicle plus 16 per
                                    slot of workspace and 16 coalesced bytes per vehicle-update;
                                    never changes the traffic (see ts_read_emissions) */
    /* Vehicle types (trucks differ "in size, acceleration, and maximum speed"; DESIGN.md
     * reading R31).  n_types == 0: one type { veh_len, a, no speed cap }.  Otherwise type t =
     * { type_len[t] >= 2 m, type_a[t] > 0 m/s^2, type_vmax[t] > 0 m/s } and veh_len / a are not used:
     * a vehicle's desired speed is min(v0_mult * edge limit, type_vmax), Eq. 7 uses its own `a`,
     * and every gap is measured to the REAR of the vehicle ahead, i.e. with that vehicle's length
     * (the atlas carries the occupant's type beside its speed code). */
    uint32_t n_types;            /* 0..4 */
    float type_len[4];
    float type_a[4];
    float type_vmax[4];
    /* Control variants (readings R34-R36). */
    uint32_t amber_steps;        /* amber after every green: a vehicle goes on iff v^2 > 2 b (C - x); 0 = none */
    float stop_dist;             /* TS_CTRL_STOP: a vehicle has made its stop once it is within stop_dist m of */
    float stop_speed;            /*   the line at no more than stop_speed m/s (both >= 0) */
    /* Re-routing (ts_reroute): route entries to reserve for each of the two route
     * tables (>= the entries of the routes given; new routes may be longer).  0 = ts_reroute is not
     * available and no workspace is spent on it (one shortest-path tree of N words per distinct
     * origin node, the graph in CSR form, 20 N bytes for each of the 592 trees in flight). */
    uint32_t route_capacity;
} ts_params;

/* Device resources lent by the caller for the lifetime of the ts_sim. */
typedef struct ts_device {
    void *workspace;          /* DEVICE pointer, 256-byte aligned */
    size_t bytes;             /* >= ts_query_workspace */
    void *cuda_stream;        /* cudaStream_t (NULL = legacy default stream) */
    int out_on_device;        /* non-zero: ts_read_* / digest outputs are device pointers */
} ts_device;

/* Length-V arrays in vehicle-id order (any pointer may be NULL), plus scalars. */
typedef struct ts_state_out {
    uint8_t *status;          /* TS_PENDING / TS_ACTIVE / TS_ARRIVED */
    uint32_t *edge;           /* current edge (first route edge while pending, last when arrived) */
    uint8_t *lane;
    uint32_t *cell;           /* floor(x) */
    float *x;                 /* m from the edge start (front bumper); == edge length once arrived */
    float *v;                 /* m/s */
    uint32_t *route_idx;      /* index into the vehicle's route */
    uint32_t *insert_step;    /* step at which it became ACTIVE (0 while pending) */
    uint32_t *arrive_step;    /* step at which it ARRIVED (0 before) */
    /* scalars, always written (host memory, whatever out_on_device says) */
    uint64_t step;
    uint32_t n_pending, n_active, n_arrived;
    uint64_t vehicle_updates; /* sum over steps of ACTIVE vehicles advanced (the bench metric) */
} ts_state_out;

/* Length-E integer accumulators (PAPER.md:437 samples; the utilisation of PAPER.md:446 is derived
 * from them by ts_read_utilisation). */
typedef struct ts_edge_stats_out {
    uint32_t *entered;               /* vehicles that entered the edge (departures included) */
    uint32_t *exited;                /* vehicles that left it (arrivals included) */
    uint64_t *exit_steps_sum;        /* sum over exits of steps spent on the edge */
    uint32_t *sample_count_sum;      /* sum over samples of vehicles on the edge */
    uint64_t *sample_speedcode_sum;  /* sum over samples and vehicles of round(4 v) (0.25 m/s units) */
    uint32_t n_samples;              /* always host */
} ts_edge_stats_out;

typedef struct ts_sim ts_sim;

/* Device bytes ts_create needs for these inputs.  Pure host arithmetic; validates sizes only. */
int ts_query_workspace(const ts_network *net, const ts_routes *routes,
                       const ts_departures *dep, const ts_params *params, size_t *bytes);

/* The inputs of the microsimulation, PAPER.md:366-374 ("the road network ... each edge contains the
 * number of lanes, the speed limit", per-vehicle departure times and procedural variables) and
 * PAPER.md:382-384 (the per-vehicle paths): validate them, lay out the workspace, copy them (H2D on
 * dev->cuda_stream) and set the state of step 0: every vehicle PENDING, the traffic atlas of
 * PAPER.md:404-406 empty.  All pointers inside the structs are HOST pointers owned by the caller; the
 * library copies what it needs and keeps none.  *out is NULL on failure.
 * Errors: TS_EINVAL (sizes, ranges, a route that is not contiguous, look-ahead or entry zone shorter
 * than one step's advance, signal cycle beyond 2^24 steps, ...), TS_ENOMEM (workspace smaller than
 * ts_query_workspace says), TS_ECUDA (no device: there is no CPU fallback).
 * The host work (validation, departure-queue index) runs on up to 16 threads; the copy of the route table, the
 * largest input, is enqueued first and overlaps it when the caller's buffer is pinned.  With the environment
 * variable TS_TRACE_CREATE set, the milliseconds of each stage go to stderr.
 * Layout of the atlas: one occupancy bit per cell and one speed-code byte per 4 cells when every vehicle length is
 * >= 4 m and insert_clear_cells >= 4 (two vehicles of a lane then never share 4 cells), else one byte per cell; the
 * environment variable TS_CODE_GRANULE=0 forces the latter (a diagnostic; results are the same, the workspace larger). */
int ts_create(const ts_network *net, const ts_routes *routes, const ts_departures *dep,
              const ts_params *params, const ts_device *dev, ts_sim **out);

/* The time-stepped simulation of PAPER.md:390 ("we simulate the traffic by updating each individual
 * vehicle: lane changing (mandatory or discretionary) and vehicle following, and update the travel
 * time, position, and velocity ... In our implementation, we use dt = 0.5 s"): enqueue n steps on the
 * stream (one step = DESIGN.md section 2, steps 1-5: signals, intent of every ACTIVE vehicle by Eq. 7
 * PAPER.md:394-397 and the lane-change / gap-acceptance rules PAPER.md:399-400, departures, claims at
 * the controls of PAPER.md:402, commit, sampling).  Asynchronous; returns TS_EINVARIANT if a sticky
 * device error was read back earlier, TS_EINVAL if the step counter would pass 2^31. */
int ts_step(ts_sim *sim, uint32_t n);

/* Same, and writes one 64-bit state digest per step to digests[0..n) (DESIGN.md section 2.6:
 * order-independent sum of SplitMix64-mixed (id, edge, lane, bits(x), bits(v)) over ACTIVE
 * vehicles plus a mix of the counters).  Synchronises when digests is a host pointer. */
int ts_step_digest(ts_sim *sim, uint32_t n, uint64_t *digests);

/* Back to step 0 without re-uploading the inputs. */
int ts_reset(ts_sim *sim);

/* Per-vehicle outputs, PAPER.md:360 ("Given we simulate individual vehicles, we can extract many
 * measurements"): a snapshot in vehicle-id order into caller-allocated arrays (HOST pointers unless
 * ts_device.out_on_device; any may be NULL) plus scalars.  Runs the device-side audit of the atlas
 * (every ACTIVE vehicle's cell is marked, exactly n_active cells are marked, no position or speed is
 * NaN, negative or infinite) and reports a violation as the sticky TS_EINVARIANT.  Synchronises. */
int ts_read_state(ts_sim *sim, ts_state_out *out);

/* Per-edge outputs, PAPER.md:437 ("we sample every minute the utilization and per edge speed"): the
 * integer accumulators since ts_create / ts_reset / the last call with reset != 0 (which zeroes them
 * after the copy).  Length-E caller-allocated arrays (HOST unless out_on_device; any may be NULL).
 * Synchronises. */
int ts_read_edge_stats(ts_sim *sim, ts_edge_stats_out *out, int reset);

/* "We defined utilization as the number of vehicles at the sampling time divided by the
 * maximum number of vehicles that can fit on the edge.  This capacity is computed as the length of the
 * edge times the number of lines divided by the average length of a vehicle plus the lead gap" --
 * utilisation[e] = (sample_count_sum[e] / n_samples) / (len_e * lanes_e / (veh_len + s0)) -- and the
 * mean sampled speed in m/s, over the samples since the last reset of the statistics
 * (reset them every 720 steps for the paper's 6-minute groups).  fp32, computed on the device; two
 * length-E arrays (HOST unless out_on_device; either may be NULL); 0 where there is no sample.
 * Synchronises. */
int ts_read_utilisation(ts_sim *sim, float *utilisation, float *mean_speed);

/* Section 6.3.4 "Vehicle energy consumption and pollution estimates".
 * Fills two caller-allocated length-V fp32 arrays in vehicle-id order (either may be NULL; HOST
 * pointers unless ts_device.out_on_device): grams of CO emitted (Eq. 8, Stein and
 * Walker 2003) and millilitres of fuel burnt (Eq. 9, Akcelik 1989) by each vehicle
 * since step 0.  Every step each ACTIVE vehicle adds rate(v_k, a_k) * dt, a_k = (v_{k+1} as
 * integrated - v_k) / dt (readings R28-R30).  Each vehicle owns its accumulators, so
 * the fp32 sums are reproducible bit for bit.  Synchronises.  TS_EINVAL unless the sim was
 * created with ts_params.emissions != 0. */
int ts_read_emissions(ts_sim *sim, float *co_g, float *fuel_ml);

/* Iterative decaying re-routing, PAPER.md:386 (section 6.3.1: "we use the microsimulation measurements
 * to update those weights and repeat the microsimulation ... we recompute all routes the first and second
 * iteration, and then we decay it to half and one-fourth of the vehicles") with PAPER.md:431 ("we replace
 * [per-vehicle Dijkstra] with ... All Pairs Shortest Path"): one shortest-path tree per distinct origin.
 * Readings R37-R41 of DESIGN.md:
 *   weights   w[e] = round-half-up(256 * exit_steps_sum[e] / exited[e]) from the statistics accumulated
 *             since the last reset (what ts_read_edge_stats shows), or w_free[e] where no vehicle has
 *             left the edge; clamped to 1..2^20; units of 1/256 simulation step; all integer.
 *   w_free    HOST array [E], 1..2^20: the caller's free-flow weights (the paper's initialisation).
 *   mask      HOST array [V] or NULL (= everybody): vehicles with mask[i] != 0 get the shortest path
 *             from the tail node of their first edge to the head node of their last edge, ties broken
 *             by taking at every node, walking back from the destination, the inbound edge with the
 *             smallest (distance, edge id); the others keep their route; so does a vehicle whose
 *             origin is its destination.
 * All on the device (weights, trees, route extraction, offsets); the host only rebuilds the index of
 * departure queues for the new first edges.  Ends with ts_reset: step 0, statistics cleared.
 * out (nullable) receives counts, device times and, if out->w != NULL, the E weights used (host pointer
 * unless ts_device.out_on_device).  Synchronises.
 * Errors: TS_EINVAL (route_capacity == 0, bad w_free, a path cost beyond 2^32), TS_ENOMEM (new routes
 * longer than route_capacity; the routes in use are then unchanged). */
typedef struct ts_reroute_out {
    uint32_t n_rerouted;      /* vehicles asked to re-route */
    uint32_t n_trees;         /* shortest-path trees computed */
    uint64_t route_entries;   /* length of the new route table */
    float sssp_ms;            /* device time of the tree kernel */
    float device_ms;          /* device time of weights + trees + extraction */
    uint32_t *w;              /* [E] or NULL */
} ts_reroute_out;
int ts_reroute(ts_sim *sim, const uint32_t *w_free, const uint8_t *mask, ts_reroute_out *out);

/* The routes in use: HOST arrays route_off [V+1] and route_edges [*n_entries] (either may be NULL;
 * call once with both NULL to learn *n_entries).  Synchronises. */
int ts_read_routes(ts_sim *sim, uint64_t *route_off, uint32_t *route_edges, uint64_t *n_entries);

/* Static user equilibrium by the Frank-Wolfe algorithm with BPR travel times -- the paper's static
 * traffic assignment model, PAPER.md:307-338 (section 5.3: steps 1-4, objective Eq. 6) with the BPR
 * curve of PAPER.md:200-216 (Eq. 3: t = t0 (1 + alpha (v/c)^beta), beta = 4).  A self-contained call
 * on the same shortest-path kernel as ts_reroute.  Readings R42-R44 of DESIGN.md: beta is the integer
 * 4; the all-or-nothing step grows its trees on integer weights max(1, rint(t * weight_scale)) with
 * the tie-break of ts_reroute; demand is integer trips per OD pair.
 * All arrays of ts_sue_problem are HOST arrays; flow / time of ts_sue_out are HOST arrays [E] unless
 * ts_device.out_on_device; objective [iterations + 1], gap and step [iterations] are always host (any
 * may be NULL).  gap[k] = (x.t - y.t) / x.t before step k (0 at equilibrium, Wardrop's condition,
 * PAPER.md:313); step[k] in [0, 1] by bisection on the derivative along the segment; objective[k] =
 * Eq. 6 at x_k.  fp64.  Synchronises.  Errors: TS_EINVAL, TS_ENOMEM (workspace), TS_ECUDA. */
typedef struct ts_sue_problem {
    uint32_t n_nodes, n_edges;
    const uint32_t *edge_from, *edge_to;   /* [E] */
    const double *t0;                      /* [E] free-flow time (Eq. 4), > 0 */
    const double *cap;                     /* [E] capacity in the demand's unit of time, > 0 */
    uint32_t n_od;
    const uint32_t *od_origin, *od_dest;   /* [n_od] nodes */
    const uint32_t *od_trips;              /* [n_od] */
    double alpha;                          /* 0.15 */
    double weight_scale;                   /* integer weight = max(1, rint(t * weight_scale)), <= 2^20 */
    uint32_t iterations;                   /* Frank-Wolfe iterations after the initial assignment */
    uint32_t bisections;                   /* of the line search, <= 64 */
} ts_sue_problem;
typedef struct ts_sue_out {
    double *flow, *time;
    double *objective, *gap, *step;
    float device_ms, sssp_ms;              /* device time of the whole solve / of the tree kernel */
    uint32_t n_trees;
} ts_sue_out;
int ts_sue_workspace(const ts_sue_problem *problem, size_t *bytes);
int ts_sue_solve(const ts_sue_problem *problem, const ts_device *dev, ts_sue_out *out);

/* Checkpoint / resume.  The workspace is the caller's, so a checkpoint is a copy of it (the step kernels' whole
 * state: slots, atlas, claims, queues, statistics, the route table in use) behind a small header with the
 * host-side counters.  ts_checkpoint_size gives the bytes, ts_checkpoint fills a HOST buffer of that size,
 * ts_restore puts a simulation created from the SAME inputs back into that state (checked: TS_EINVAL if the
 * layout differs or the buffer is not a checkpoint); stepping on from there gives bit for bit what the
 * uninterrupted run gives.  Tuning options (ts_set_option) are not part of it.  Both calls synchronise. */
int ts_checkpoint_size(ts_sim *sim, size_t *bytes);
int ts_checkpoint(ts_sim *sim, void *host_buf);
int ts_restore(ts_sim *sim, const void *host_buf);

/* Shortest-path trees WITHOUT ANY ALLOCATION, for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it): the tree kernel of ts_reroute / ts_sue_solve
 * (readings R37-R38) with its scratch -- per tree in flight a 64-bit label, two frontier words and
 * a stamp per node -- in a file-scope static device array of 20 MiB that every GPU loading this library holds
 * until the process exits.  Limit: n_nodes <= ts_sssp_static_max_nodes() = 65 536 (beyond it: TS_EINVAL and a
 * message; use the workspace-based calls).  The call allocates nothing on device or host, copies nothing and
 * does not synchronise: it enqueues ONE kernel on cuda_stream.
 * ALL pointers are DEVICE pointers owned by the caller:
 *   d_out_off [n_nodes+1], d_out_edge [n_edges]   CSR of the outbound edges by tail node (edge ids)
 *   d_edge_to [n_edges]  head nodes;  d_w [n_edges]  integer weights in 1..2^20
 *   d_sources [n_sources]  source nodes;  d_pred [n_sources * n_nodes]  OUT: row i = tree of d_sources[i], per
 *                        node the inbound edge on the shortest path (ties: smallest (distance, edge id)),
 *                        0xFFFFFFFF at the source and at unreachable nodes
 *   d_error (nullable)   one word the caller has zeroed; set to 1 if a path cost passed 2^32
 * The static array is shared by every call on the GPU and keeps the last call's contents (nothing needs
 * clearing: the kernel initialises a tree's labels and stamps before growing it).  Calls that OVERLAP on the GPU
 * (two streams without a dependency) race on it: order them. */
uint32_t ts_sssp_static_max_nodes(void);
int ts_sssp_static(uint32_t n_nodes, uint32_t n_edges, const uint32_t *d_out_off, const uint32_t *d_out_edge,
                   const uint32_t *d_edge_to, const uint32_t *d_w, const uint32_t *d_sources, uint32_t n_sources,
                   uint32_t *d_pred, uint32_t *d_error, void *cuda_stream);

/* Tuning knobs that never change results.
 *  "mode"          1 (default) = ts_step(n) is ONE persistent cooperative kernel looping over
 *                  the n steps with grid-wide barriers; 0 = one launch per phase.
 *  "threads"       CTA size of the persistent kernel (multiple of 32 in 64..1024).  Default: not
 *                  fixed -- ts_step enqueues every chunk of 2048 steps twice, with 640 threads
 *                  (spill-free; best while a step is one warp's latency) and with 768 (more warps;
 *                  best once a CTA holds several rounds of vehicles), and the device runs the one
 *                  that fits the number of live slots; the other launch returns at once.  Setting
 *                  "threads" or "blocks_per_sm" (or "profile") fixes the size; "adaptive" 1 undoes it.
 *  "adaptive_chunk", "adaptive_above", "adaptive_big"  steps per chunk (default 2048), the number of live slots
 *                  above which the big size is preferred (default 640 per SM; -1 restores it), and the big
 *                  size itself (0 = the default: 768).
 *  "blocks_per_sm" resident CTAs per SM of the persistent kernel (default 1).
 *  "sort_period"   steps between compaction of retired slots + re-sort of the live ones by
 *                  edge; 0 = never; default 128 (256 on networks
 *                  with more than 4 M sort keys).
 *  "sort_groups"   the re-sort key is (vehicle id & (sort_groups - 1), edge): a power of two between 1 (by edge
 *                  alone) and the lane-change period when that is a power of two <= 8 (the default: whole
 *                  warps then take or skip the lane-change code together).
 *  "smem_tiles"    most tiles (one vehicle per thread) whose move records the persistent kernel keeps in
 *                  shared memory; the rest go through L2.  Shared memory and L1 share one array per
 *                  SM: what the records leave stays L1 for the edge records.  Default 6.
 *  "profile"       non-zero: the persistent kernel clocks its phases (see ts_read_profile). */
int ts_set_option(ts_sim *sim, const char *key, long long value);

/* Option "profile": out[0..5] = nanoseconds (GPU global timer, mean over the CTAs) spent in
 * phase 1 (until the whole CTA is done), waiting at the barrier after it, phase 2, the barrier
 * after it, compaction + re-sort, and the digest, summed over out[6] steps since ts_create /
 * ts_reset.  out[7] = the largest per-CTA phase-1 total of one ts_step call.  Host array.
 * Synchronises. */
int ts_read_profile(ts_sim *sim, uint64_t out[8]);

/* Frees host bookkeeping only; the workspace stays the caller's. */
void ts_destroy(ts_sim *sim);

/* Thread-local message of the last non-zero return. */
const char *ts_last_error(void);
/* "major.minor (build flags)" */
const char *ts_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TRAFFICSIM_H */
