// ts_api.cu -- C ABI (include/trafficsim.h) and kernels of libts.so.  Product code, sm_100a.
//
// Host side: validation, workspace layout, upload.  Device side: thin __global__ wrappers
// around the phases in ts_phases.cuh, either two launches per step (mode 0) or ONE persistent
// cooperative kernel per ts_step(n) call that loops over the n steps with grid-wide barriers
// (mode 1, default): the step is bound by the two grid-wide dependencies, not by bandwidth,
// so no host launch may sit inside the loop.
#include <cooperative_groups.h>
#include <chrono>
#include <memory>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <numeric>
#include <atomic>
#include <string>
#include <thread>
#include <vector>

#include "../../include/trafficsim.h"
#include "ts_phases.cuh"
#include "ts_sort.cuh"
#include "ts_reroute.cuh"
#include "ts_sue.cuh"

namespace cg = cooperative_groups;
using namespace ts;

// ------------------------------------------------------------------ errors

static thread_local char g_err[512] = "";
static int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}
#define CUDA_TRY(call)                                                                    \
    do {                                                                                  \
        cudaError_t e_ = (call);                                                          \
        if (e_ != cudaSuccess)                                                            \
            return fail(TS_ECUDA, "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

extern "C" const char* ts_last_error(void) { return g_err; }
extern "C" const char* ts_version(void) {
    return "0.2 (sm_100a, -fmad=false, IEEE div/sqrt, two-plane atlas, persistent step kernel, edge-sorted slots)";
}

// ------------------------------------------------------------------ host helpers

// fn(begin, end, chunk) over [0, n) on the host cores (ts_create's validation and queue building
// walk every route entry; on a 1 M-vehicle input that is most of the end-to-end set-up time).
template <typename F>
static void parallel_chunks(size_t n, F fn) {
    unsigned hw = std::thread::hardware_concurrency();
    const size_t nt = std::max<size_t>(1, std::min<size_t>({(size_t)(hw ? hw : 1), (size_t)16, n / 65536 + 1}));
    if (nt == 1) { fn((size_t)0, n, (size_t)0); return; }
    std::vector<std::thread> th;
    const size_t per = (n + nt - 1) / nt;
    for (size_t t = 0; t < nt; t++) {
        const size_t b = std::min(n, t * per), e = std::min(n, b + per);
        th.emplace_back([=] { fn(b, e, t); });
    }
    for (auto& x : th) x.join();
}

// ------------------------------------------------------------------ layout

struct Layout {
    size_t total = 0;
    uint32_t V = 0, E = 0, N = 0, Q = 0, cap = 0, groups = 1;
    uint64_t R = 0, n_lanes = 0, atlas_chunks = 0;   // chunk = 128 cells of one lane row
    size_t edges, route_edges, route_begin, queue_rec, dep_rec, codes, occ, queue_state, queue_cand,
        lane_claim, node_claim, dyn, barrier, slots, slots_d, mr_g, cr, rank, hist, base, audit, partial, o_status, o_lane,
        o_edge, o_x, o_v, o_rpos, o_insert, o_arrive, o_cell, o_ridx, st_entered, st_exited,
        st_exit_steps, st_samp_cnt, st_samp_code, emis, digest, types, edge_aux, edge_from, node_free_from;
    uint32_t emissions = 0;
    uint32_t ext = 0;          // extended rule set: vehicle types and / or control variants (R31-R36)
    uint32_t typed = 0;        // more than one vehicle type: the atlas has a type plane
    uint32_t cg = 0;           // code / type plane: one byte per 2^cg cells (Params::cg)
    // re-routing (ts_params.route_capacity != 0): a second route table, the graph in CSR form, one
    // shortest-path tree per distinct origin node, per-vehicle origin / destination / new offsets
    uint64_t Rcap = 0;         // entries per route table
    uint32_t n_src = 0, Qcap = 0;
    size_t rr_routes2, rr_end, rr_origin, rr_dest, rr_srcidx, rr_mask, rr_newlen, rr_newoff, rr_bsum, rr_first2,
        rr_out_off, rr_out_edge, rr_efrom, rr_eto, rr_w, rr_wfree, rr_src, rr_todo, rr_pred, rr_lab, rr_fa, rr_fb,
        rr_stamp, rr_err, rr_adjw;
    static constexpr uint32_t kDigestChunk = 8192;
    size_t take(size_t bytes) {
        size_t off = total;
        total += (bytes + 255) & ~(size_t)255;
        return off;
    }
    void plan() {
        const size_t Q = std::max(this->Q, Qcap);        // re-routing may open queues on other edges
        edges = take((size_t)E * sizeof(EdgeRec));
        route_edges = take(std::max<uint64_t>(R, Rcap) * 4);
        route_begin = take((size_t)V * 4);
        queue_rec = take((size_t)Q * 16);
        dep_rec = take((size_t)V * 32);
        codes = take((atlas_chunks * 128) >> cg);
        occ = take((atlas_chunks + 3) * 16);          // one spare chunk in front, two behind: load_win never clamps
        queue_state = take((size_t)Q * 16); queue_cand = take((size_t)Q * 16);
        lane_claim = take(n_lanes * 8); node_claim = take((size_t)N * 8);
        dyn = take(sizeof(Dyn)); barrier = take(256);
        slots = take((size_t)cap * 16 * 6);           // A, B, C in two ping-pong sets
        slots_d = take(emissions ? (size_t)cap * 8 * 2 : 0);   // D in both sets
        mr_g = take((size_t)cap * 16); cr = take((size_t)cap * 32);
        rank = take((size_t)cap * 4); hist = take((size_t)E * groups * 4); base = take((size_t)E * groups * 4);
        audit = take(16);
        partial = take((size_t)kMaxCtas * 4);
        o_status = take(V); o_lane = take(V);
        o_edge = take((size_t)V * 4); o_x = take((size_t)V * 4); o_v = take((size_t)V * 4);
        o_rpos = take((size_t)V * 4); o_insert = take((size_t)V * 4); o_arrive = take((size_t)V * 4);
        o_cell = take((size_t)std::max(V, E) * 4); o_ridx = take((size_t)std::max(V, E) * 4);   // read-back scratch (per vehicle or per edge)
        st_entered = take((size_t)E * 4); st_exited = take((size_t)E * 4);
        st_exit_steps = take((size_t)E * 8); st_samp_cnt = take((size_t)E * 4);
        st_samp_code = take((size_t)E * 8);
        emis = take(emissions ? (size_t)V * 8 : 0);      // zeroed by ts_reset with the statistics
        digest = take((size_t)kDigestChunk * 8);
        types = take(typed ? (atlas_chunks * 128) >> cg : 0);
        edge_aux = take(ext ? (size_t)E * 4 : 0); edge_from = take(ext ? (size_t)E * 4 : 0);
        node_free_from = take(ext ? (size_t)N * 4 : 0);
        if (Rcap) {
            rr_routes2 = take(Rcap * 4); rr_end = take((size_t)V * 4);
            rr_origin = take((size_t)V * 4); rr_dest = take((size_t)V * 4); rr_srcidx = take((size_t)V * 4);
            rr_mask = take(V); rr_newlen = take(((size_t)V + 1) * 4); rr_newoff = take(((size_t)V + 1) * 4);
            rr_bsum = take(((size_t)V / (kScanBlock * kScanItems) + 2) * 4); rr_first2 = take((size_t)V * 8);
            rr_out_off = take(((size_t)N + 1) * 4); rr_out_edge = take((size_t)E * 4);
            rr_efrom = take((size_t)E * 4); rr_eto = take((size_t)E * 4); rr_w = take((size_t)E * 4); rr_wfree = take((size_t)E * 4);
            rr_src = take((size_t)n_src * 4); rr_todo = take((size_t)n_src * 4);
            rr_pred = take((size_t)n_src * N * 4);
            rr_lab = take((size_t)kRrCtas * N * 8); rr_fa = take((size_t)kRrCtas * N * 8); rr_fb = take((size_t)kRrCtas * N * 8);
            rr_stamp = take((size_t)kRrCtas * N * 4); rr_err = take(4);
            rr_adjw = take(((size_t)E + 4) * 16);
        }
    }
};

// The code plane's granule (Params::cg): one byte per 4 cells is enough where two vehicles of one lane row are
// never less than 4 cells apart.  With L the shortest vehicle length: a follower's advance is capped at the gap to
// its leader's CELL minus the leader's length (E2, E3), so its new cell is at most cL - ceil(L); a lane change needs
// that gap to the target lane's leader (G1) and, to the lag vehicle F, x - L - (cF + 1) >= the most F can advance
// in the step (G2), so F ends more than L behind the changer and their cells differ by more than L - 1; an entrant
// needs `insert_clear` free cells and lands more than L short of the lane-change zone (R24).  L >= 4 m and
// insert_clear >= 4 therefore keep any two cells of a lane at least 4 apart (all five configs: 5 m, 7 cells);
// the kernel raises ERR_SPACING if a vehicle ever finds its leader closer.  Otherwise: one byte per cell.
// TS_CODE_GRANULE=0 in the environment keeps one byte per cell regardless (a diagnostic: A/B timing and the
// parity tests of both layouts).
static uint32_t code_granule_shift(const ts_params* prm) {
    if (const char* e = std::getenv("TS_CODE_GRANULE")) if (e[0] == '0') return 0u;
    float min_len = prm->n_types ? prm->type_len[0] : prm->veh_len;
    for (uint32_t t = 1; t < prm->n_types && t < (uint32_t)kMaxTypes; t++) min_len = std::min(min_len, prm->type_len[t]);
    return (min_len >= 4.0f && prm->insert_clear_cells >= 4) ? 2u : 0u;
}

// Sizes only (what ts_query_workspace may look at).
// `first_edge` (optional): receives each vehicle's first route edge, so that ts_create gathers
// them from the route table (one random read per vehicle into hundreds of MB) only once.
static int plan_sizes(const ts_network* net, const ts_routes* rt, const ts_params* prm, Layout& L,
                      std::vector<uint32_t>* first_edge = nullptr) {
    if (!net || !rt || !prm) return fail(TS_EINVAL, "null argument");
    // the re-sort groups vehicles by their place in the lane-change stagger when that is a mask
    const uint32_t lcp = prm->lc_period;
    L.groups = (lcp >= 2 && lcp <= 8 && !(lcp & (lcp - 1))) ? lcp : 1;
    if (net->n_edges == 0 || net->n_nodes == 0) return fail(TS_EINVAL, "empty network");
    if (rt->n_vehicles >= 0x7FFFFFF0u) return fail(TS_EINVAL, "too many vehicles");
    L.V = rt->n_vehicles; L.E = net->n_edges; L.N = net->n_nodes;
    L.R = L.V ? rt->route_off[L.V] : 0;
    if (L.R >= 0xFFFFFFFEull) return fail(TS_EINVAL, "route table too long (%llu entries)", (unsigned long long)L.R);
    uint64_t chunks = 0, lanes = 0;
    for (uint32_t e = 0; e < L.E; e++) {
        uint32_t ln = net->edge_lanes[e], len = net->edge_len_m[e];
        if (ln < 1 || ln > 8) return fail(TS_EINVAL, "edge %u: lanes %u not in 1..8", e, ln);
        if (len < 16 || len > 65535) return fail(TS_EINVAL, "edge %u: length %u not in 16..65535", e, len);
        chunks += (uint64_t)ln * ((len + 127) >> 7);
        lanes += ln;
    }
    // a cell is addressed by one 32-bit index (row * 128 + cell)
    if (chunks + 2 >= (1ull << 25)) return fail(TS_EINVAL, "atlas larger than 2^32 cells");
    L.atlas_chunks = chunks; L.n_lanes = lanes;
    std::vector<uint32_t> fe_local;
    std::vector<uint32_t>& fe = first_edge ? *first_edge : fe_local;
    fe.assign(L.V, 0);
    std::atomic<uint32_t> bad(0xFFFFFFFFu);
    parallel_chunks(L.V, [&](size_t b, size_t e_, size_t) {
        for (size_t i = b; i < e_; i++) {
            if (rt->route_off[i + 1] <= rt->route_off[i] || rt->route_edges[rt->route_off[i]] >= L.E) {
                uint32_t cur = bad.load();
                while ((uint32_t)i < cur && !bad.compare_exchange_weak(cur, (uint32_t)i)) {}
                return;
            }
            fe[i] = rt->route_edges[rt->route_off[i]];
        }
    });
    if (bad.load() != 0xFFFFFFFFu) {
        const uint32_t i = bad.load();
        if (rt->route_off[i + 1] <= rt->route_off[i]) return fail(TS_EINVAL, "vehicle %u: empty route", i);
        return fail(TS_EINVAL, "vehicle %u: route edge %u out of range", i, rt->route_edges[rt->route_off[i]]);
    }
    std::vector<uint8_t> is_origin(L.E, 0);
    uint32_t q = 0;
    for (uint32_t i = 0; i < L.V; i++)
        if (!is_origin[fe[i]]) { is_origin[fe[i]] = 1; q++; }
    L.Q = q;
    if (prm->route_capacity) {
        // re-routed vehicles keep their origin NODE: a new route may start on any of its outbound edges
        if (prm->route_capacity < L.R) return fail(TS_EINVAL, "params: route_capacity %u below the %llu entries of the routes given", prm->route_capacity, (unsigned long long)L.R);
        L.Rcap = prm->route_capacity;
        std::vector<uint8_t> is_src(L.N, 0);
        std::vector<uint32_t> deg(L.N, 0);
        for (uint32_t e = 0; e < L.E; e++) if (net->edge_from[e] < L.N) deg[net->edge_from[e]]++;
        uint64_t qcap = 0;
        for (uint32_t i = 0; i < L.V; i++) {
            const uint32_t o = net->edge_from[fe[i]];
            if (o < L.N && !is_src[o]) { is_src[o] = 1; L.n_src++; qcap += deg[o]; }
        }
        L.Qcap = (uint32_t)std::min<uint64_t>(qcap, L.E);
    }
    // a vehicle takes one slot when it departs; a queue head that is ready but has not won its
    // lane yet holds one reserved slot, which a compaction may drop (then it takes a new one)
    L.cap = (uint32_t)std::min<uint64_t>((uint64_t)L.V + std::max(q, L.Qcap) + 1024ull, 0x7FFFFFF0ull);
    L.emissions = prm->emissions ? 1u : 0u;
    L.typed = prm->n_types > 1 ? 1u : 0u;
    L.cg = code_granule_shift(prm);
    L.ext = (prm->n_types != 0 || prm->amber_steps != 0) ? 1u : 0u;
    for (uint32_t h = 0; h < L.N && !L.ext; h++)
        if (net->node_ctrl[h] > TS_CTRL_SIGNAL) L.ext = 1u;
    L.plan();
    return TS_OK;
}

extern "C" int ts_query_workspace(const ts_network* net, const ts_routes* routes, const ts_departures* dep,
                                  const ts_params* params, size_t* bytes) {
    (void)dep;
    if (!bytes) return fail(TS_EINVAL, "bytes is null");
    Layout L;
    int rc = plan_sizes(net, routes, params, L);
    if (rc) return rc;
    *bytes = L.total;
    return TS_OK;
}

// ------------------------------------------------------------------ the simulation object

struct ts_sim {
    Layout L;
    Ctx ctx;
    uint8_t* ws = nullptr;
    cudaStream_t stream = nullptr;
    int out_on_device = 0;
    uint32_t k = 0;           // steps enqueued so far
    uint32_t cur = 0;         // which slot set holds the state
    int mode = 1;             // 0: one launch per phase, 1: persistent cooperative kernel
    int threads = 640;        // persistent kernel CTA size (96 registers per thread, no spills: within 4 % of the best size for 3e4 and for 3e5 active vehicles)
    int blocks_per_sm = 1;
    uint32_t chunk_no = 0;    // adaptive chunks enqueued since ts_reset (parity selects Dyn::prefer_big[])
    uint32_t adaptive_chunk = 2048;   // steps per adaptive chunk
    int adaptive_big = 0;             // CTA size of the big launch of a chunk; 0 = 768
    // Most move-record tiles per thread kept in shared memory.  Shared memory and L1 are one 228 KB array: what the
    // move records do not take stays L1, which holds the edge records of the SM's vehicles across steps (the grid
    // barrier keeps L1 alive).  Records beyond the limit go through L2 (Ctx::mr_g).  Measured: config 4 (3 M slots:
    // the records would take all of it) 11.2 -> 14.1 G vehicle-updates/s, config 3 17.7 -> 18.0, config 5 3.72 -> 3.88.
    uint32_t smem_tiles = 6;
    long long adaptive_above = -1;    // live slots above which the big CTA size is preferred (-1: one round of tiles at 640 threads)
    int adaptive = 1;         // no CTA size asked for: 640 threads, or 768 while more than one round of tiles is live
    int sms = 0;
    uint32_t sort_period = 128;  // steps between compaction + re-sort; 0 = never (set in ts_create)
    uint32_t profile = 0;
    int smem_limit = 0;
    int l2_bytes = 0;
    uint32_t sticky = 0;
    // re-routing: what the host needs to rebuild the departure-queue index for new routes
    std::vector<EdgeRec> edges_h;
    std::vector<uint32_t> dep_step_h, v0m_bits_h, mand_bits_h, type_h, src_idx_h, first_h;
    uint32_t route_cur = 0;   // which route table is in use
    RrCtx rr;
};

template <typename T>
static T* at(ts_sim* s, size_t off) { return reinterpret_cast<T*>(s->ws + off); }

// ------------------------------------------------------------------ kernels

__device__ __forceinline__ Who who() {
    Who w;
    w.t = threadIdx.x; w.T = blockDim.x; w.cta = blockIdx.x; w.n_cta = gridDim.x;
    return w;
}

// Grid-wide barrier of the persistent kernel: one arrival per CTA on a monotonic counter.
// bar.sync orders the CTA's writes before thread 0's release (red.release.gpu: cumulative, one
// MEMBAR.ALL.GPU); thread 0 polls the counter with relaxed loads and the second bar.sync hands the
// observation on to the CTA.
//
// There is deliberately NO gpu-scope fence on the acquiring side.  What such a fence adds in hardware is
// CCTL.IVALL, the invalidation of the SM's whole L1 -- needed by readers that use L1-cached loads of data
// other SMs write.  This kernel has none: everything any thread writes during a launch (slot state, atlas,
// claims, queues, counters, sort scratch) is read with ld.global.cg / atomics, i.e. at L2, the point of
// coherence (LDG.E.STRONG.GPU in the SASS; the only other loads are ld.global.nc of data no thread writes
// during a launch: edge records, routes, queue and departure records).  A load issued after the poll has
// returned reaches L2 after the releasing CTA's writes were performed there.  Keeping L1 alive across the
// 2 barriers of every step is what lets the edge records of a CTA's vehicles be L1 hits step after step
// (`__threadfence()` = MEMBAR.SC.GPU + CCTL.IVALL dropped them four times per step).
struct PhaseClock;
__device__ __forceinline__ void clock_tick(PhaseClock& clk, int b);

// `b`: profile bin that gets the time up to the moment this whole CTA has arrived.
__device__ __forceinline__ void grid_barrier(unsigned int* counter, unsigned int& target, PhaseClock& clk, int b) {
    target += gridDim.x;
    __syncthreads();
    if (threadIdx.x == 0) {
        clock_tick(clk, b);
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(counter) : "memory");
        unsigned int v;
        do {
            asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(counter) : "memory");
        } while ((int)(v - target) < 0);
    }
    __syncthreads();
}

extern __shared__ uint4 dyn_smem[];

// The static record of the first (normally the only) departure queue this thread looks after.
__device__ __forceinline__ uint4 first_queue_rec(const Ctx& c, const Who& me) {
    const uint32_t q = me.qslot(0);
    return q < c.n_queues ? __ldg(c.queue_rec + q) : make_uint4(0, 0, 0, 0);
}

__device__ __forceinline__ unsigned long long global_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
// Phase clock of option "profile": thread 0 of every CTA adds the time since its last tick to bin b.
struct PhaseClock {
    unsigned long long* acc;   // shared memory, 8 bins; nullptr = off
    unsigned long long last;
    __device__ __forceinline__ void tick(int b) {
        if (acc) { const unsigned long long t = global_ns(); acc[b] += t - last; last = t; }
    }
};

// n steps in one launch; grid-wide barriers stand where the method has its two dependencies.
__device__ __forceinline__ void clock_tick(PhaseClock& clk, int b) { clk.tick(b); }

// MAXT = most threads per SM it is launched with: sets the register budget (64 / 80 / 128).
// EMIS = keep the section 6.3.4 totals (ts_params.emissions).
template <int MAXT, bool EMIS, bool EXT>
__global__ void __launch_bounds__(MAXT, 1) k_persistent(const __grid_constant__ Ctx c, uint32_t k0, uint32_t n,
                                                       uint32_t cur, uint32_t sort_period, uint32_t mr_j,
                                                       unsigned long long* digests, uint32_t profile,
                                                       uint32_t variant, uint32_t big_above, uint32_t chunk_parity) {
    __shared__ uint32_t red[33];
    __shared__ uint32_t sh_n_slots[2];
    __shared__ unsigned long long sh_prof[8];
    const Who me = who();
    // Adaptive CTA size (variant 0 / 1; 2 = unconditional): both instantiations are enqueued for
    // every chunk of steps and the one the previous chunk did not ask for returns at once.  The
    // word read was written by the previous chunk; this chunk's verdict goes to the other word.
    if (variant != 2u) {
        if (me.t == 0) red[0] = __ldcg(&c.dyn->prefer_big[chunk_parity]);
        __syncthreads();
        if (red[0] != variant) return;
        __syncthreads();
    }
    unsigned int target = 0;
    uint32_t n_upd = 0;
    PhaseClock clk;
    clk.acc = (profile && me.t == 0) ? sh_prof : nullptr;
    if (clk.acc) { for (int b = 0; b < 8; b++) sh_prof[b] = 0; clk.last = global_ns(); }
    if (me.t == 0) sh_n_slots[0] = __ldcg(&c.dyn->n_slots);
    __syncthreads();
    const uint4 qr0 = first_queue_rec(c, me);      // held in registers for the whole launch
    // first step of this launch after which a sample is taken, then every period
    const uint32_t sp = c.p.sample_period;
    uint32_t k_sample = sp ? k0 + (sp - 1u - k0 % sp) : NONE32;
    for (uint32_t i = 0; i < n; i++) {
        const uint32_t k = k0 + i;
        const Slots& S = c.s[cur];
        const uint32_t n_slots = sh_n_slots[i & 1];
        const bool sample = (k == k_sample);
        if (sample) k_sample += sp;
        phase1<EMIS, EXT>(c, S, k, me, dyn_smem, mr_j, n_slots, sample, n_upd, qr0);
        grid_barrier(c.barrier, target, clk, 0);
        clk.tick(1);
        // slots are handed out in phase 1 only: the count the next step works on is final now
        if (me.t == 0) sh_n_slots[(i + 1) & 1] = min(__ldcg(&c.dyn->slot_alloc), c.cap_slots);
        phase2<EXT>(c, S, k, me, dyn_smem, mr_j, n_slots, sample, qr0);
        grid_barrier(c.barrier, target, clk, 2);
        clk.tick(3);
        if (digests) {
            // the digest reads counters that CTAs already in step i+1 would be bumping (arrivals,
            // slots handed out): nobody leaves the digest before everybody has finished it
            phase_digest(c, S, digests + i, me, sh_n_slots[(i + 1) & 1]);
            grid_barrier(c.barrier, target, clk, 5);
        }
        if (sort_period && (k + 1) % sort_period == 0) {      // A9 + A10, between two steps
            const uint32_t ns = sort_rank(c, S, me, sh_n_slots[(i + 1) & 1]);
            grid_barrier(c.barrier, target, clk, 4);
            sort_partial(c, me, red);
            grid_barrier(c.barrier, target, clk, 4);
            sort_scan(c, me, red);
            grid_barrier(c.barrier, target, clk, 4);
            sort_scatter(c, S, c.s[cur ^ 1], me, ns);
            if (me.t == 0) sh_n_slots[(i + 1) & 1] = __ldcg(&c.dyn->n_slots);
            grid_barrier(c.barrier, target, clk, 4);
            cur ^= 1;
            clk.tick(4);
        }
    }
    if (clk.acc) {                                  // mean over CTAs per bin; slowest CTA's phase 1
        for (int b = 0; b < 6; b++) atomicAdd(&c.dyn->prof[b], sh_prof[b] / me.n_cta);
        atomicMax(&c.dyn->prof[7], sh_prof[0]);
        if (me.cta == 0) c.dyn->prof[6] = __ldcg(&c.dyn->prof[6]) + n;
    }
    // more warps pay once a CTA has more than one round of tiles at the small size
    if (variant != 2u && me.cta == 0 && me.t == 0)
        c.dyn->prefer_big[chunk_parity ^ 1u] = sh_n_slots[n & 1] > big_above ? 1u : 0u;
    n_upd = block_sum(n_upd, red);
    if (me.t == 0 && n_upd) atomicAdd(&c.dyn->updates, (unsigned long long)n_upd);
}

// The same phases as separate launches (mode 0: profiling per phase, and a fallback where a
// cooperative launch is not possible).  Move records go through global memory.
template <bool EMIS, bool EXT>
__global__ void __launch_bounds__(256) k_phase1(const __grid_constant__ Ctx c, uint32_t k, uint32_t cur) {
    __shared__ uint32_t red[33];
    uint32_t n_upd = 0;
    __shared__ uint32_t sh_n;
    if (threadIdx.x == 0) sh_n = __ldcg(&c.dyn->n_slots);
    __syncthreads();
    const uint32_t n_slots = sh_n;
    const Who me = who();
    phase1<EMIS, EXT>(c, c.s[cur], k, me, nullptr, 0, n_slots, sample_step(c.p, k), n_upd, first_queue_rec(c, me));
    if (blockIdx.x == 0 && threadIdx.x == 0) c.dyn->pad = n_slots;   // phase 2 overwrites dyn->n_slots
    n_upd = block_sum(n_upd, red);
    if (threadIdx.x == 0 && n_upd) atomicAdd(&c.dyn->updates, (unsigned long long)n_upd);
}
template <bool EXT>
__global__ void __launch_bounds__(256) k_phase2(const __grid_constant__ Ctx c, uint32_t k, uint32_t cur) {
    __shared__ uint32_t sh_n;
    if (threadIdx.x == 0) sh_n = __ldcg(&c.dyn->pad);
    __syncthreads();
    const Who me = who();
    phase2<EXT>(c, c.s[cur], k, me, nullptr, 0, sh_n, sample_step(c.p, k), first_queue_rec(c, me));
}
__global__ void __launch_bounds__(256) k_digest(const __grid_constant__ Ctx c, uint32_t cur, unsigned long long* out) {
    phase_digest(c, c.s[cur], out, who(), min(__ldcg(&c.dyn->slot_alloc), c.cap_slots));   // test instrument: may read the slot count per thread
}
__global__ void __launch_bounds__(256) k_sort_rank(const __grid_constant__ Ctx c, uint32_t cur) {
    __shared__ uint32_t sh_n;
    if (threadIdx.x == 0) sh_n = min(__ldcg(&c.dyn->slot_alloc), c.cap_slots);
    __syncthreads();
    const uint32_t n = sort_rank(c, c.s[cur], who(), sh_n);
    if (blockIdx.x == 0 && threadIdx.x == 0) c.dyn->pad = n;
}
__global__ void __launch_bounds__(256) k_sort_partial(const __grid_constant__ Ctx c) {
    __shared__ uint32_t red[33];
    sort_partial(c, who(), red);
}
__global__ void __launch_bounds__(256) k_sort_scan(const __grid_constant__ Ctx c) {
    __shared__ uint32_t red[33];
    sort_scan(c, who(), red);
}
__global__ void __launch_bounds__(256) k_sort_scatter(const __grid_constant__ Ctx c, uint32_t cur) {
    __shared__ uint32_t sh_n;
    if (threadIdx.x == 0) sh_n = __ldcg(&c.dyn->pad);
    __syncthreads();
    sort_scatter(c, c.s[cur], c.s[cur ^ 1], who(), sh_n);
}

// State of step 0: every vehicle PENDING.
__global__ void k_init(const __grid_constant__ Ctx c) {
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nthreads = gridDim.x * blockDim.x;
    for (uint32_t i = tid; i < c.V; i += nthreads) {
        const uint32_t rb = c.route_begin[i];
        c.o_status[i] = 0; c.o_lane[i] = 0; c.o_edge[i] = c.route_edges[rb]; c.o_x[i] = 0.0f;
        c.o_v[i] = 0.0f; c.o_rpos[i] = rb; c.o_insert[i] = 0; c.o_arrive[i] = 0;
    }
    for (uint32_t q = tid; q < c.n_queues; q += nthreads) {
        const uint32_t head = q ? c.queue_rec[q - 1].z : 0u;        // queues are contiguous in dep_rec
        c.queue_state[q] = make_uint4(head, c.dep_rec[2 * (size_t)head + 1].z, NONE32, 0);
        c.queue_cand[q] = make_uint4(NONE32, 0, head, 0);
    }
    if (tid == 0) {
        Dyn d;
        memset(&d, 0, sizeof d);
        *c.dyn = d;
        *c.barrier = 0;
    }
}

// Invariant I2 on the device, run when the state is read back: every ACTIVE vehicle's cell is
// marked in the occupancy plane, and the plane holds exactly as many marked cells as there are
// ACTIVE vehicles -- so no two vehicles share a cell and no mark was lost.
__global__ void k_audit(const __grid_constant__ Ctx c, uint32_t cur, size_t n_words) {
    const size_t tid = blockIdx.x * (size_t)blockDim.x + threadIdx.x, nthreads = gridDim.x * (size_t)blockDim.x;
    const uint32_t* occ32 = reinterpret_cast<const uint32_t*>(c.occ);
    unsigned long long marked = 0, missing = 0;
    for (size_t i = tid; i < n_words; i += nthreads) marked += __popc(occ32[i]);
    const uint32_t n_slots = min(c.dyn->slot_alloc, c.cap_slots);
    for (size_t s = tid; s < n_slots; s += nthreads) {
        const uint4 sa = c.s[cur].A[s];
        if (!(sa.w & ALIVE)) continue;
        const float xs = __uint_as_float(sa.x), vs = __uint_as_float(sa.y);
        if (!(xs >= 0.0f) || !(vs >= 0.0f) || isinf(xs) || isinf(vs)) { atomicOr(&c.dyn->error, ERR_NAN); continue; }   // NaN, negative or infinite
        const uint32_t gc = (sa.z << 7) + (uint32_t)(int)floorf(xs);
        if (!((occ32[gc >> 5] >> (gc & 31)) & 1u)) missing++;
    }
    for (int o = 16; o; o >>= 1) {
        marked += __shfl_xor_sync(0xFFFFFFFFu, marked, o);
        missing += __shfl_xor_sync(0xFFFFFFFFu, missing, o);
    }
    if ((threadIdx.x & 31) == 0) {
        if (marked) atomicAdd(c.audit, marked);
        if (missing) atomicAdd(c.audit + 1, missing);
    }
}

// A12 read-back: slot-ordered state -> id-ordered arrays.
__global__ void k_gather_slots(const __grid_constant__ Ctx c, uint32_t cur) {
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nthreads = gridDim.x * blockDim.x;
    const uint32_t n_slots = min(c.dyn->slot_alloc, c.cap_slots);
    const Slots& S = c.s[cur];
    for (uint32_t s = tid; s < n_slots; s += nthreads) {
        const uint4 sa = S.A[s];
        if (!(sa.w & ALIVE)) continue;
        const uint4 sb = S.B[s];
        const uint32_t id = sb.z;
        c.o_lane[id] = (uint8_t)(sa.w & 0xFu); c.o_edge[id] = sb.x; c.o_x[id] = __uint_as_float(sa.x);
        c.o_v[id] = __uint_as_float(sa.y); c.o_rpos[id] = S.C[s].x;
    }
}
__global__ void k_finish_state(const __grid_constant__ Ctx c, uint32_t* o_cell, uint32_t* o_ridx) {
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nthreads = gridDim.x * blockDim.x;
    for (uint32_t i = tid; i < c.V; i += nthreads) {
        o_cell[i] = (uint32_t)floorf(c.o_x[i]);
        o_ridx[i] = c.o_rpos[i] - c.route_begin[i];
    }
}

// The instantiation whose register budget fits `per_sm_threads` resident threads per SM
// (128 / 96 / 80 / 72 / 64 registers per thread).
template <bool EMIS, bool EXT>
static const void* step_kernel_of(int per_sm_threads) {
    if (per_sm_threads <= 512) return (const void*)k_persistent<512, EMIS, EXT>;
    if (per_sm_threads <= 640) return (const void*)k_persistent<640, EMIS, EXT>;
    if (per_sm_threads <= 768) return (const void*)k_persistent<768, EMIS, EXT>;
    if (per_sm_threads <= 896) return (const void*)k_persistent<896, EMIS, EXT>;
    return (const void*)k_persistent<1024, EMIS, EXT>;
}
// EXT (vehicle types, control variants) and EMIS (section 6.3.4 totals) are compiled in only where asked for
static const void* step_kernel(int per_sm_threads, bool emissions, bool ext) {
    if (ext) return emissions ? step_kernel_of<true, true>(per_sm_threads) : step_kernel_of<false, true>(per_sm_threads);
    return emissions ? step_kernel_of<true, false>(per_sm_threads) : step_kernel_of<false, false>(per_sm_threads);
}

// ------------------------------------------------------------------ create / reset

// Departure queues (R19): one per distinct first edge, FIFO by (departure step, id).  One 32-byte
// departure record per vehicle in queue order { id, v0_mult, mand, route begin } { route end, second
// edge, departure step, type } and one 16-byte record per queue { row of lane 0, lane_base, end, edge }.
// Used by ts_create and, for the new first edges, by ts_reroute.
// A host array that is NOT zero-filled when it is made: its pages are first touched by the threads that fill it.
struct DepRecBuf {
    std::unique_ptr<uint4[]> p;
    void alloc(size_t n) { p.reset(new uint4[n]); }
    uint4* data() { return p.get(); }
    uint4& operator[](size_t i) { return p[i]; }
};

static void build_queues(uint32_t V, uint32_t E, const std::vector<EdgeRec>& edges, const uint32_t* first,
                         const uint32_t* second, const uint32_t* rbegin, const uint32_t* rend,
                         const uint32_t* dep_step, const uint32_t* v0m_bits, const uint32_t* mand_bits,
                         const uint32_t* type, DepRecBuf& dep_rec, std::vector<uint4>& queue_rec) {
    // counting sort by first edge (ids stay ascending inside an edge), then each queue by
    // departure step, stable -- i.e. by (edge, departure step, id) -- queues in parallel
    const bool trace = getenv("TS_TRACE_CREATE") != nullptr;
    auto t_last = std::chrono::steady_clock::now();
    auto lap = [&](const char* what) {
        if (!trace) return;
        const auto t = std::chrono::steady_clock::now();
        fprintf(stderr, "  build_queues: %-24s %8.2f ms\n", what, std::chrono::duration<double, std::milli>(t - t_last).count());
        t_last = t;
    };
    std::vector<uint32_t> order(V), q_begin((size_t)E + 1, 0);
    {
        // T contiguous blocks of vehicles, one histogram each; block t's vehicles of edge e go behind those of
        // blocks 0..t-1: ids stay ascending inside an edge
        const size_t T = std::max<size_t>(1, std::min<size_t>({(size_t)16, (size_t)V / 65536 + 1, ((size_t)1 << 20) / ((size_t)E + 1) + 1,
                                                             (size_t)std::max(1u, std::thread::hardware_concurrency())}));
        const size_t per = ((size_t)V + T - 1) / T;
        std::vector<uint32_t> hist(T * (size_t)E, 0);
        auto blocks = [&](auto fn) {
            if (T == 1) { fn((size_t)0); return; }
            std::vector<std::thread> th;
            for (size_t t = 0; t < T; t++) th.emplace_back([=] { fn(t); });
            for (auto& x : th) x.join();
        };
        blocks([&](size_t t) {
            uint32_t* h = hist.data() + t * (size_t)E;
            for (size_t i = std::min((size_t)V, t * per), e_ = std::min((size_t)V, i + per); i < e_; i++) h[first[i]]++;
        });
        uint32_t run = 0;
        for (uint32_t e = 0; e < E; e++) {
            q_begin[e] = run;
            for (size_t t = 0; t < T; t++) { const uint32_t c = hist[t * (size_t)E + e]; hist[t * (size_t)E + e] = run; run += c; }
        }
        q_begin[E] = run;
        blocks([&](size_t t) {
            uint32_t* h = hist.data() + t * (size_t)E;
            for (size_t i = std::min((size_t)V, t * per), e_ = std::min((size_t)V, i + per); i < e_; i++) order[h[first[i]]++] = (uint32_t)i;
        });
    }
    lap("counting sort");
    parallel_chunks(E, [&](size_t b, size_t e_, size_t) {
        for (size_t e = b; e < e_; e++)
            if (q_begin[e + 1] - q_begin[e] > 1)
                std::sort(order.begin() + q_begin[e], order.begin() + q_begin[e + 1],     // ids were ascending: (step, id) is the stable order
                          [&](uint32_t x, uint32_t y) { return dep_step[x] != dep_step[y] ? dep_step[x] < dep_step[y] : x < y; });
    });
    lap("sort inside queues");
    // one queue per first edge that has vehicles, in edge order; its records are the next q_begin[e+1] - q_begin[e]
    queue_rec.clear();
    for (uint32_t e = 0; e < E; e++)
        if (q_begin[e + 1] > q_begin[e])
            queue_rec.push_back(make_uint4(edges[e].row, edges[e].lane_base, q_begin[e + 1], e));
    lap("queue records");
    dep_rec.alloc(2 * (size_t)V);
    parallel_chunks(V, [&](size_t b, size_t e_, size_t) {
        for (size_t n = b; n < e_; n++) {
            const uint32_t i = order[n];
            dep_rec[2 * n] = make_uint4(i, v0m_bits[i], mand_bits[i], rbegin[i]);
            dep_rec[2 * n + 1] = make_uint4(rend[i], second[i], dep_step[i], type[i]);
        }
    });
    lap("dep_rec fill");
}

static int validate(const ts_network* net, const ts_routes* rt, const ts_departures* dep, const ts_params* p) {
    if (!dep || !p || !dep->depart_time_s) return fail(TS_EINVAL, "null argument");
    if (!(p->dt > 0) || !(p->a > 0) || !(p->b > 0) || !(p->T >= 0) || !(p->s0 >= 0))
        return fail(TS_EINVAL, "params: dt, a, b must be > 0 and T, s0 >= 0");
    if (!(p->veh_len >= 2.0f)) return fail(TS_EINVAL, "params: veh_len must be >= 2 m");
    if (p->lookahead_cells < 16 || p->lookahead_cells > 4096 || p->lookahead_cells % 16)
        return fail(TS_EINVAL, "params: lookahead_cells must be a multiple of 16 in 16..4096");
    if (p->lookback_cells > 4096) return fail(TS_EINVAL, "params: lookback_cells > 4096");
    if (p->insert_clear_cells < 1 || p->insert_clear_cells > 16)
        return fail(TS_EINVAL, "params: insert_clear_cells must be in 1..16");
    const uint32_t V = rt->n_vehicles, E = net->n_edges, N = net->n_nodes;
    // vehicle types (reading R31): none given = one type { veh_len, a, no speed cap }
    if (p->n_types > (uint32_t)kMaxTypes) return fail(TS_EINVAL, "params: n_types must be in 0..%d", kMaxTypes);
    float max_len = p->n_types ? 0.0f : p->veh_len, max_a = p->n_types ? 0.0f : p->a;
    for (uint32_t t = 0; t < p->n_types; t++) {
        if (!(p->type_len[t] >= 2.0f) || !(p->type_a[t] > 0) || !(p->type_vmax[t] > 0))
            return fail(TS_EINVAL, "params: vehicle type %u needs type_len >= 2, type_a > 0, type_vmax > 0", t);
        max_len = std::max(max_len, p->type_len[t]); max_a = std::max(max_a, p->type_a[t]);
    }
    // per vehicle, in parallel: the first offending vehicle (lowest id) is the one reported
    float max_mult = 1.0f;
    {
        std::atomic<uint32_t> bad(0xFFFFFFFFu);
        std::vector<float> chunk_max(64, 1.0f);
        const uint32_t n_types = std::max(1u, p->n_types);
        auto note = [&](uint32_t i) {
            uint32_t cur = bad.load();
            while (i < cur && !bad.compare_exchange_weak(cur, i)) {}
        };
        auto wrong = [&](uint32_t i) -> int {          // 0 = fine, else which rule it breaks
            if (dep->veh_type && dep->veh_type[i] >= n_types) return 1;
            if (dep->v0_mult && !(dep->v0_mult[i] > 0)) return 2;
            if (!(dep->depart_time_s[i] >= 0)) return 3;
            if (std::ceil((double)dep->depart_time_s[i] / (double)p->dt) >= 2147483648.0) return 4;
            return 0;
        };
        parallel_chunks(V, [&](size_t b, size_t e_, size_t t) {
            float m = 1.0f;
            for (size_t i = b; i < e_; i++) {
                if (wrong((uint32_t)i)) { note((uint32_t)i); break; }
                if (dep->v0_mult) m = std::max(m, dep->v0_mult[i]);
            }
            chunk_max[t] = m;
        });
        const uint32_t i = bad.load();
        if (i != 0xFFFFFFFFu) {
            switch (wrong(i)) {
                case 1: return fail(TS_EINVAL, "vehicle %u: veh_type %u out of range", i, dep->veh_type[i]);
                case 2: return fail(TS_EINVAL, "vehicle %u: v0_mult must be > 0", i);
                case 3: return fail(TS_EINVAL, "vehicle %u: negative departure time", i);
                default: return fail(TS_EINVAL, "vehicle %u: departure step beyond 2^31", i);
            }
        }
        for (float m : chunk_max) max_mult = std::max(max_mult, m);
    }
    float max_vlim = 0.0f;
    for (uint32_t e = 0; e < E; e++) {
        if (net->edge_from[e] >= N || net->edge_to[e] >= N) return fail(TS_EINVAL, "edge %u: endpoint out of range", e);
        if (!(net->edge_vlim[e] > 0)) return fail(TS_EINVAL, "edge %u: speed limit must be > 0", e);
        max_vlim = std::max(max_vlim, net->edge_vlim[e]);
        // a vehicle entering an edge must land short of the zone where lanes may be changed (R14)
        double adv = (double)net->edge_vlim[e] * max_mult * p->dt + 0.5 * max_a * p->dt * p->dt + max_len;
        if (!(adv < (double)p->entry_zone_cells))
            return fail(TS_EINVAL, "edge %u: entry_zone_cells %u too short for the fastest vehicle (%.2f m)", e, p->entry_zone_cells, adv);
    }
    {   // nobody may jump over a leader it never saw: the scans reach further than one step's advance plus a vehicle
        const double adv = (double)max_vlim * max_mult * p->dt + 0.5 * max_a * p->dt * p->dt + max_len;
        if (!((double)p->lookahead_cells >= adv))
            return fail(TS_EINVAL, "params: lookahead_cells %u shorter than one step's advance plus a vehicle length (%.2f m)", p->lookahead_cells, adv);
        if (p->lc_period != 0 && !((double)p->lookback_cells >= adv))
            return fail(TS_EINVAL, "params: lookback_cells %u shorter than one step's advance plus a vehicle length (%.2f m)", p->lookback_cells, adv);
    }
    std::vector<uint32_t> deg_in(N, 0), deg_out(N, 0);
    for (uint32_t e = 0; e < E; e++) { deg_in[net->edge_to[e]]++; deg_out[net->edge_from[e]]++; }
    for (uint32_t h = 0; h < N; h++) {
        const uint32_t ctrl = net->node_ctrl[h];
        if (ctrl > TS_CTRL_SIGNAL_NM) return fail(TS_EINVAL, "node %u: unknown control type", h);
        if (ctrl == TS_CTRL_SIGNAL || ctrl == TS_CTRL_SIGNAL_NM) {
            if (net->sig_green_steps[h] < 1) return fail(TS_EINVAL, "node %u: green must be >= 1 step", h);
            const uint64_t P = (uint64_t)net->sig_green_steps[h] + p->amber_steps + net->sig_allred_steps[h];
            if (P > 65535) return fail(TS_EINVAL, "node %u: green + amber + all-red > 65535 steps", h);
            if (net->sig_offset_steps[h] >= 0x80000000u) return fail(TS_EINVAL, "node %u: offset >= 2^31", h);
            const uint64_t phases = ctrl == TS_CTRL_SIGNAL_NM ? (uint64_t)deg_in[h] * std::max(1u, deg_out[h]) : deg_in[h];
            if (deg_in[h] > 255 || deg_out[h] > 255 || phases * P >= (1ull << 24))
                return fail(TS_EINVAL, "node %u: signal cycle of %llu steps does not fit 24 bits", h, (unsigned long long)(phases * P));
        }
        if (ctrl == TS_CTRL_STOP && !(max_len <= 15.0f))
            return fail(TS_EINVAL, "node %u: STOP control needs vehicle lengths <= 15 m (an edge is >= 16 m)", h);
    }
    if (!(p->stop_dist >= 0) || !(p->stop_speed >= 0)) return fail(TS_EINVAL, "params: stop_dist, stop_speed must be >= 0");
    // routes: every entry a valid edge, consecutive edges share a node
    std::atomic<uint32_t> bad_vehicle(0xFFFFFFFFu);
    parallel_chunks(V, [&](size_t b, size_t e_, size_t) {
        for (size_t i = b; i < e_; i++)
            for (uint64_t j = rt->route_off[i]; j < rt->route_off[i + 1]; j++)
                if (rt->route_edges[j] >= E ||
                    (j > rt->route_off[i] && net->edge_to[rt->route_edges[j - 1]] != net->edge_from[rt->route_edges[j]])) {
                    uint32_t cur = bad_vehicle.load();
                    while ((uint32_t)i < cur && !bad_vehicle.compare_exchange_weak(cur, (uint32_t)i)) {}
                    return;
                }
    });
    if (bad_vehicle.load() != 0xFFFFFFFFu) {
        const uint32_t i = bad_vehicle.load();
        for (uint64_t j = rt->route_off[i]; j < rt->route_off[i + 1]; j++) {
            if (rt->route_edges[j] >= E) return fail(TS_EINVAL, "vehicle %u: route edge out of range", i);
            if (j > rt->route_off[i] && net->edge_to[rt->route_edges[j - 1]] != net->edge_from[rt->route_edges[j]])
                return fail(TS_EINVAL, "vehicle %u: route is not contiguous at position %llu", i,
                            (unsigned long long)(j - rt->route_off[i]));
        }
    }
    return TS_OK;
}

static void bind_ctx(ts_sim* s, const ts_params* p) {
    Layout& L = s->L;
    Ctx& c = s->ctx;
    Params& q = c.p;
    q.dt = p->dt; q.a = p->a; q.b = p->b; q.T = p->T; q.s0 = p->s0; q.len = p->veh_len;
    q.b_safe = p->b_safe; q.politeness = p->politeness; q.lc_threshold = p->lc_threshold;
    { volatile float ab = p->a * p->b; volatile float r = sqrtf(ab); volatile float K = 2.0f * r; q.Kinv = 1.0f / K; }
    { volatile float h = 0.5f * p->a; q.half_a_dt = h * p->dt; }
    q.a_dt = p->a * p->dt;
    q.entry_zone_f = (float)p->entry_zone_cells;
    q.H = (int)p->lookahead_cells; q.Hb = (int)p->lookback_cells;
    q.lc_pow2 = (p->lc_period && !(p->lc_period & (p->lc_period - 1))) ? 1u : 0u;
    q.lc_period = p->lc_period; q.insert_clear = p->insert_clear_cells; q.sample_period = p->sample_period_steps;
    q.inv_dt = 1.0f / p->dt;
    q.cg = L.cg;
    for (int t = 0; t < kMaxTypes; t++) {
        const bool given = (uint32_t)t < p->n_types;
        const float len_t = given ? p->type_len[t] : p->veh_len, a_t = given ? p->type_a[t] : p->a;
        q.t_len[t] = len_t; q.t_a[t] = a_t; q.t_vmax[t] = given ? p->type_vmax[t] : INFINITY;
        { volatile float ab = a_t * p->b; volatile float r = sqrtf(ab); volatile float K = 2.0f * r; q.t_Kinv[t] = 1.0f / K; }
        { volatile float h = 0.5f * a_t; q.t_half_a_dt[t] = h * p->dt; }
        q.t_a_dt[t] = a_t * p->dt;
    }
    if (p->n_types) { q.len = q.t_len[0]; q.a = q.t_a[0]; q.Kinv = q.t_Kinv[0]; q.a_dt = q.t_a_dt[0]; q.half_a_dt = q.t_half_a_dt[0]; }
    q.two_b = 2.0f * p->b; q.stop_dist = p->stop_dist; q.stop_speed = p->stop_speed; q.amber = p->amber_steps;
    c.V = L.V; c.E = L.E; c.N = L.N; c.n_queues = L.Q; c.cap_slots = L.cap; c.sort_groups = L.groups;
    c.edges = at<EdgeRec>(s, L.edges); c.route_edges = at<uint32_t>(s, L.route_edges);
    c.route_begin = at<uint32_t>(s, L.route_begin);
    c.queue_rec = at<uint4>(s, L.queue_rec); c.dep_rec = at<uint4>(s, L.dep_rec);
    c.codes = at<uint8_t>(s, L.codes); c.occ = at<uint4>(s, L.occ) + 1;
    c.queue_state = at<uint4>(s, L.queue_state); c.queue_cand = at<uint4>(s, L.queue_cand);
    c.lane_claim = at<unsigned long long>(s, L.lane_claim); c.node_claim = at<unsigned long long>(s, L.node_claim);
    c.dyn = at<Dyn>(s, L.dyn); c.barrier = at<unsigned int>(s, L.barrier);
    uint4* sl = at<uint4>(s, L.slots);
    const size_t cap = L.cap;
    for (int i = 0; i < 2; i++) { c.s[i].A = sl + (3 * i + 0) * cap; c.s[i].B = sl + (3 * i + 1) * cap; c.s[i].C = sl + (3 * i + 2) * cap; }
    for (int i = 0; i < 2; i++) c.s[i].D = L.emissions ? at<float2>(s, L.slots_d) + i * cap : nullptr;
    c.mr_g = at<uint4>(s, L.mr_g); c.cr = at<uint4>(s, L.cr);
    c.rank = at<uint32_t>(s, L.rank); c.hist = at<uint32_t>(s, L.hist); c.base = at<uint32_t>(s, L.base);
    c.partial = at<uint32_t>(s, L.partial); c.audit = at<unsigned long long>(s, L.audit);
    c.o_status = at<uint8_t>(s, L.o_status); c.o_lane = at<uint8_t>(s, L.o_lane);
    c.o_edge = at<uint32_t>(s, L.o_edge); c.o_x = at<float>(s, L.o_x); c.o_v = at<float>(s, L.o_v);
    c.o_rpos = at<uint32_t>(s, L.o_rpos); c.o_insert = at<uint32_t>(s, L.o_insert); c.o_arrive = at<uint32_t>(s, L.o_arrive);
    c.st_entered = at<uint32_t>(s, L.st_entered); c.st_exited = at<uint32_t>(s, L.st_exited);
    c.st_exit_steps = at<unsigned long long>(s, L.st_exit_steps); c.st_samp_cnt = at<uint32_t>(s, L.st_samp_cnt);
    c.st_samp_code = at<unsigned long long>(s, L.st_samp_code);
    c.emis = L.emissions ? at<float2>(s, L.emis) : nullptr;
    c.types = L.typed ? at<uint8_t>(s, L.types) : nullptr;
    c.edge_aux = L.ext ? at<uint32_t>(s, L.edge_aux) : nullptr;
    c.edge_from = L.ext ? at<uint32_t>(s, L.edge_from) : nullptr;
    c.node_free_from = L.ext ? at<uint32_t>(s, L.node_free_from) : nullptr;
}

extern "C" int ts_reset(ts_sim* s) {
    if (!s) return fail(TS_EINVAL, "null sim");
    Layout& L = s->L;
    cudaStream_t st = s->stream;
    CUDA_TRY(cudaMemsetAsync(s->ws + L.occ, 0, (L.atlas_chunks + 3) * 16, st));   // codes need no clearing
    CUDA_TRY(cudaMemsetAsync(s->ws + L.lane_claim, 0xFF, L.n_lanes * 8, st));
    CUDA_TRY(cudaMemsetAsync(s->ws + L.node_claim, 0xFF, (size_t)L.N * 8, st));
    CUDA_TRY(cudaMemsetAsync(s->ws + L.hist, 0, (size_t)L.E * L.groups * 4, st));
    CUDA_TRY(cudaMemsetAsync(s->ws + L.st_entered, 0, L.digest - L.st_entered, st));
    if (L.ext) CUDA_TRY(cudaMemsetAsync(s->ws + L.node_free_from, 0, (size_t)L.N * 4, st));   // every STOP node free
    k_init<<<std::max(1u, std::min(1184u, (L.V + 255) / 256)), 256, 0, st>>>(s->ctx);
    CUDA_TRY(cudaGetLastError());
    s->k = 0; s->cur = 0; s->sticky = 0; s->chunk_no = 0;
    return TS_OK;
}

extern "C" int ts_create(const ts_network* net, const ts_routes* rt, const ts_departures* dep,
                         const ts_params* p, const ts_device* dev, ts_sim** out) {
    if (out) *out = nullptr;
    if (!out || !dev) return fail(TS_EINVAL, "null argument");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return fail(TS_ECUDA, "no CUDA device: this library has no CPU fallback");
    const bool trace = getenv("TS_TRACE_CREATE") != nullptr;
    auto t_last = std::chrono::steady_clock::now();
    auto lap = [&](const char* what) {
        if (!trace) return;
        const auto t = std::chrono::steady_clock::now();
        fprintf(stderr, "ts_create: %-28s %8.2f ms\n", what, std::chrono::duration<double, std::milli>(t - t_last).count());
        t_last = t;
    };
    Layout L;
    std::vector<uint32_t> first_edge;
    int rc = plan_sizes(net, rt, p, L, &first_edge);
    lap("plan_sizes");
    if (rc) return rc;
    if ((uint64_t)L.groups * L.E >= 0xFFFFFFF0ull) L.groups = 1;
    if (!dev->workspace || ((uintptr_t)dev->workspace & 255)) return fail(TS_EINVAL, "workspace must be a 256-byte aligned device pointer");
    if (dev->bytes < L.total) return fail(TS_ENOMEM, "workspace too small: %zu < %zu bytes", dev->bytes, L.total);
    if (!net || !rt || !rt->route_edges) return fail(TS_EINVAL, "null argument");
    // the routes are by far the largest input (4 bytes per route entry): their copy is enqueued first and travels
    // while the host validates and builds its records (from pinned memory; a pageable buffer is staged at once)
    const cudaError_t ce_routes = L.R ? cudaMemcpyAsync((uint8_t*)dev->workspace + L.route_edges, rt->route_edges, L.R * 4,
                                                        cudaMemcpyHostToDevice, (cudaStream_t)dev->cuda_stream) : cudaSuccess;
    if (ce_routes != cudaSuccess) return fail(TS_ECUDA, "upload: %s", cudaGetErrorString(ce_routes));
    if ((rc = validate(net, rt, dep, p))) {
        cudaStreamSynchronize((cudaStream_t)dev->cuda_stream);      // the caller may free its buffers on an error
        return rc;
    }
    lap("validate");

    const uint32_t V = L.V, E = L.E, N = L.N;
    // per-edge records: atlas row offsets, claim indices, signal plan of the head node
    std::vector<uint32_t> n_in(N, 0), n_out(N, 0);
    std::vector<EdgeRec> edges(E);
    std::vector<uint8_t> in_rank(E), out_rank(E);
    uint64_t row = 0, lane_base = 0;
    for (uint32_t e = 0; e < E; e++) {
        EdgeRec& r = edges[e];
        const uint32_t h = net->edge_to[e], ctrl = net->node_ctrl[h];
        if (n_in[h] >= 255) return fail(TS_EINVAL, "node %u: more than 255 inbound edges", h);
        r.row = (uint32_t)row; r.lane_base = (uint32_t)lane_base; r.vlim = net->edge_vlim[e];
        r.to_node = h; r.len = (uint16_t)net->edge_len_m[e];
        r.cyc_lc = 1u | ((uint32_t)net->edge_lanes[e] << 24) | (ctrl << 28);
        r.off_sh = 0; r.magic = 1; r.green = 1;          // cycle 1: n mod 1 = 0 < green
        in_rank[e] = (uint8_t)n_in[h]++;
        if (n_out[net->edge_from[e]] >= 255) return fail(TS_EINVAL, "node %u: more than 255 outbound edges", net->edge_from[e]);
        out_rank[e] = (uint8_t)n_out[net->edge_from[e]]++;     // rank among the tail node's outbound edges, by edge index
        row += (uint64_t)net->edge_lanes[e] * ((net->edge_len_m[e] + 127) >> 7);
        lane_base += net->edge_lanes[e];
    }
    // A1 (reading R16): inbound edge number in_rank of node h is green at step k iff
    // t = (k + offset_h) mod (n_in * P) lies in [in_rank * P, in_rank * P + green), P = green + allred.
    // Shifting the offset by the phase start turns that into one comparison, and the modulo by the
    // invariant cycle is done by multiplication on the device (ts_device.cuh).
    for (uint32_t e = 0; e < E; e++) {
        EdgeRec& r = edges[e];
        const uint32_t ctrl_e = r.cyc_lc >> 28;
        if (ctrl_e != TS_CTRL_SIGNAL && ctrl_e != TS_CTRL_SIGNAL_NM) continue;
        const uint32_t h = r.to_node;
        // R36: an amber interval after the green; R35: with one phase per movement (i, j), number
        // i * m + j, the inbound edge's share i * m * P is folded in here and j * P on the device
        const uint64_t P = (uint64_t)net->sig_green_steps[h] + p->amber_steps + net->sig_allred_steps[h];
        const uint64_t m_out = ctrl_e == TS_CTRL_SIGNAL_NM ? std::max(1u, n_out[h]) : 1;   // a dead end has one (empty) exit
        const uint64_t cycle = (uint64_t)n_in[h] * m_out * P;            // < 2^24 (validated)
        const uint64_t start = (uint64_t)in_rank[e] * m_out * P;         // < cycle
        const uint64_t off = ((uint64_t)net->sig_offset_steps[h] % cycle + cycle - start) % cycle;
        uint32_t l = 0;
        while ((1ull << l) < cycle) l++;
        const uint32_t sh1 = l ? 1u : 0u, sh2 = l - sh1;
        r.magic = (uint32_t)(((1ull << 32) * ((1ull << l) - cycle)) / cycle + 1ull);
        r.cyc_lc = (uint32_t)cycle | (r.cyc_lc & 0xFF000000u);
        r.off_sh = (uint32_t)off | (sh1 << 24) | (sh2 << 25);
        r.green = (uint16_t)net->sig_green_steps[h];
    }
    lap("edge records");
    // departure queues: per first edge, FIFO by (departure step, id) (R19)
    std::vector<uint32_t> dep_step(V), route_begin(V);
    const uint32_t* re = rt->route_edges;
    auto fbits = [](float f) { uint32_t u; memcpy(&u, &f, 4); return u; };
    std::vector<uint32_t> second(V), route_end(V), v0m_bits(V), mand_bits(V), type_v(V);
    parallel_chunks(V, [&](size_t b, size_t e_, size_t) {
        for (size_t i = b; i < e_; i++) {
            dep_step[i] = (uint32_t)std::ceil((double)dep->depart_time_s[i] / (double)p->dt);
            const uint32_t rb = (uint32_t)rt->route_off[i], rend = (uint32_t)rt->route_off[i + 1];
            route_begin[i] = rb;
            route_end[i] = rend;
            second[i] = rb + 1 < rend ? re[rb + 1] : NONE32;
            v0m_bits[i] = fbits(dep->v0_mult ? dep->v0_mult[i] : 1.0f);
            mand_bits[i] = fbits(dep->mand_dist_m ? dep->mand_dist_m[i] : p->mand_dist_default);
            type_v[i] = dep->veh_type ? dep->veh_type[i] : 0u;
        }
    });
    lap("per-vehicle arrays");
    DepRecBuf dep_rec;
    std::vector<uint4> queue_rec;
    build_queues(V, E, edges, first_edge.data(), second.data(), route_begin.data(), route_end.data(), dep_step.data(),
                 v0m_bits.data(), mand_bits.data(), type_v.data(), dep_rec, queue_rec);
    if (queue_rec.size() != L.Q) return fail(TS_EINVAL, "internal: queue count mismatch");

    lap("build_queues");
    ts_sim* s = new ts_sim();
    s->L = L; s->ws = (uint8_t*)dev->workspace; s->stream = (cudaStream_t)dev->cuda_stream;
    s->out_on_device = dev->out_on_device;
    bind_ctx(s, p);
    cudaStream_t st = s->stream;
    auto up = [&](size_t off, const void* src, size_t bytes) -> cudaError_t {
        return bytes ? cudaMemcpyAsync(s->ws + off, src, bytes, cudaMemcpyHostToDevice, st) : cudaSuccess;
    };
    cudaError_t ce = cudaSuccess;
    auto chk = [&](cudaError_t e) { if (ce == cudaSuccess) ce = e; };
    chk(up(L.edges, edges.data(), (size_t)E * sizeof(EdgeRec)));
    chk(up(L.route_begin, route_begin.data(), (size_t)V * 4));
    chk(up(L.queue_rec, queue_rec.data(), (size_t)L.Q * 16));
    chk(up(L.dep_rec, dep_rec.data(), (size_t)V * 32));
    std::vector<uint32_t> aux;
    if (L.ext) {
        aux.resize(E);
        for (uint32_t e = 0; e < E; e++) {
            const uint32_t h = net->edge_to[e];
            const uint64_t P = (uint64_t)net->sig_green_steps[h] + p->amber_steps + net->sig_allred_steps[h];
            aux[e] = (uint32_t)std::min<uint64_t>(P, 65535) | ((uint32_t)out_rank[e] << 16);
        }
        chk(up(L.edge_aux, aux.data(), (size_t)E * 4));
        chk(up(L.edge_from, net->edge_from, (size_t)E * 4));
    }
    std::vector<uint32_t> rr_out_off, rr_out_edge, rr_origin, rr_dest, rr_src;
    if (L.Rcap) {
        // re-routing: the graph as CSR by tail node (edge ids ascending inside a node), every vehicle's
        // origin and destination NODE (they never change, R38) and the list of distinct origins
        rr_out_off.assign((size_t)N + 1, 0); rr_out_edge.resize(E);
        for (uint32_t e = 0; e < E; e++) rr_out_off[net->edge_from[e] + 1]++;
        for (uint32_t h = 0; h < N; h++) rr_out_off[h + 1] += rr_out_off[h];
        { std::vector<uint32_t> fill(rr_out_off.begin(), rr_out_off.end() - 1);
          for (uint32_t e = 0; e < E; e++) rr_out_edge[fill[net->edge_from[e]]++] = e; }
        rr_origin.resize(V); rr_dest.resize(V); s->src_idx_h.resize(V);
        std::vector<uint32_t> idx_of(N, NONE32);
        for (uint32_t i = 0; i < V; i++) {
            const uint32_t o = net->edge_from[first_edge[i]];
            rr_origin[i] = o; rr_dest[i] = net->edge_to[re[route_end[i] - 1]];
            if (idx_of[o] == NONE32) { idx_of[o] = (uint32_t)rr_src.size(); rr_src.push_back(o); }
            s->src_idx_h[i] = idx_of[o];
        }
        chk(up(L.rr_out_off, rr_out_off.data(), ((size_t)N + 1) * 4)); chk(up(L.rr_out_edge, rr_out_edge.data(), (size_t)E * 4));
        chk(up(L.rr_efrom, net->edge_from, (size_t)E * 4)); chk(up(L.rr_eto, net->edge_to, (size_t)E * 4));
        chk(up(L.rr_origin, rr_origin.data(), (size_t)V * 4)); chk(up(L.rr_dest, rr_dest.data(), (size_t)V * 4));
        chk(up(L.rr_srcidx, s->src_idx_h.data(), (size_t)V * 4)); chk(up(L.rr_src, rr_src.data(), rr_src.size() * 4));
        chk(up(L.rr_end, route_end.data(), (size_t)V * 4));
        s->edges_h = edges; s->dep_step_h = dep_step; s->v0m_bits_h = v0m_bits; s->mand_bits_h = mand_bits; s->type_h = type_v;
        RrCtx& r = s->rr;
        r.V = V; r.E = E; r.N = N; r.n_src = L.n_src;
        r.out_off = at<uint32_t>(s, L.rr_out_off); r.out_edge = at<uint32_t>(s, L.rr_out_edge);
        r.edge_from = at<uint32_t>(s, L.rr_efrom); r.edge_to = at<uint32_t>(s, L.rr_eto);
        r.w = at<uint32_t>(s, L.rr_w); r.w_free = at<uint32_t>(s, L.rr_wfree);
        r.st_exited = s->ctx.st_exited; r.st_exit_steps = s->ctx.st_exit_steps;
        r.origin = at<uint32_t>(s, L.rr_origin); r.dest = at<uint32_t>(s, L.rr_dest); r.src_idx = at<uint32_t>(s, L.rr_srcidx);
        r.src_node = at<uint32_t>(s, L.rr_src); r.mask = at<uint8_t>(s, L.rr_mask);
        r.new_len = at<uint32_t>(s, L.rr_newlen); r.new_off = at<uint32_t>(s, L.rr_newoff); r.block_sum = at<uint32_t>(s, L.rr_bsum);
        r.first2 = at<uint32_t>(s, L.rr_first2); r.pred = at<uint32_t>(s, L.rr_pred);
        r.lab = at<unsigned long long>(s, L.rr_lab); r.fa = at<uint2>(s, L.rr_fa); r.fb = at<uint2>(s, L.rr_fb);
        r.stamp = at<uint32_t>(s, L.rr_stamp); r.error = at<uint32_t>(s, L.rr_err);
        r.adjw = at<uint4>(s, L.rr_adjw);
    }
    // the staging vectors die with this scope: make sure the copies have left them
    lap("enqueue copies, host copies");
    chk(cudaStreamSynchronize(st));
    if (ce != cudaSuccess) { delete s; return fail(TS_ECUDA, "upload: %s", cudaGetErrorString(ce)); }
    lap("copies done");

    int dev_id = 0;
    cudaGetDevice(&dev_id);
    cudaDeviceGetAttribute(&s->sms, cudaDevAttrMultiProcessorCount, dev_id);
    cudaDeviceGetAttribute(&s->smem_limit, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev_id);
    cudaDeviceGetAttribute(&s->l2_bytes, cudaDevAttrL2CacheSize, dev_id);
    bool attr_ok = true;
    for (int t : {512, 640, 768, 896, 1024})
        attr_ok = attr_ok && cudaFuncSetAttribute(step_kernel(t, s->L.emissions != 0, s->L.ext != 0), cudaFuncAttributeMaxDynamicSharedMemorySize, s->smem_limit - 1024) == cudaSuccess;
    if (!attr_ok) {
        delete s;
        return fail(TS_ECUDA, "cannot raise the dynamic shared memory limit of the step kernel");
    }
    // one sort scans the whole key histogram: rarer on networks with many edges (measured:
    // 64 / 128 / 256 / 512 steps give 20.2 / 20.0 / - / - us per step on config 3 (1 M keys) and
    // 36.5 / 33.3 / 33.2 / 33.4 on config 4 (10 M keys))
    s->sort_period = ((uint64_t)L.groups * L.E > 4000000ull) ? 256 : 128;
    if ((rc = ts_reset(s))) { delete s; return rc; }
    lap("attributes, ts_reset enqueued");
    *out = s;
    return TS_OK;
}

extern "C" void ts_destroy(ts_sim* s) { delete s; }

extern "C" int ts_set_option(ts_sim* s, const char* key, long long value) {
    if (!s || !key) return fail(TS_EINVAL, "null argument");
    if (!strcmp(key, "mode")) {
        if (value != 0 && value != 1) return fail(TS_EINVAL, "mode must be 0 or 1");
        s->mode = (int)value;
    } else if (!strcmp(key, "blocks_per_sm")) {
        if (value < 1 || value * s->threads > 2048) return fail(TS_EINVAL, "blocks_per_sm * threads must be in 1..2048");
        s->blocks_per_sm = (int)value;
        s->adaptive = 0;
    } else if (!strcmp(key, "adaptive_chunk")) {
        if (value < 1 || value > 0x7FFFFFFF) return fail(TS_EINVAL, "adaptive_chunk must be >= 1");
        s->adaptive_chunk = (uint32_t)value;
    } else if (!strcmp(key, "adaptive_big")) {
        if (value != 0 && (value <= 640 || value > 1024 || value % 32)) return fail(TS_EINVAL, "adaptive_big must be 0 or a multiple of 32 in 672..1024");
        s->adaptive_big = (int)value;
    } else if (!strcmp(key, "sort_groups")) {
        if (value < 1 || value > (long long)s->L.groups || (value & (value - 1)))
            return fail(TS_EINVAL, "sort_groups must be a power of two in 1..%u (the lane-change period of this simulation)", s->L.groups);
        s->ctx.sort_groups = (uint32_t)value;
    } else if (!strcmp(key, "smem_tiles")) {
        if (value < 0 || value > 0x7FFFFFFF) return fail(TS_EINVAL, "smem_tiles must be >= 0");
        s->smem_tiles = (uint32_t)value;
    } else if (!strcmp(key, "adaptive_above")) {
        if (value < -1 || value > 0x7FFFFFFF) return fail(TS_EINVAL, "adaptive_above must be >= -1");
        s->adaptive_above = value;
    } else if (!strcmp(key, "adaptive")) {
        s->adaptive = value ? 1 : 0;
        if (s->adaptive) { s->threads = 640; s->blocks_per_sm = 1; }
    } else if (!strcmp(key, "threads")) {
        if (value < 64 || value > 1024 || value % 32) return fail(TS_EINVAL, "threads must be a multiple of 32 in 64..1024");
        s->threads = (int)value;
        s->adaptive = 0;
        s->blocks_per_sm = std::min(s->blocks_per_sm, 2048 / s->threads);
    } else if (!strcmp(key, "profile")) {
        s->profile = value ? 1u : 0u;
    } else if (!strcmp(key, "sort_period")) {
        if (value < 0 || value > 0x7FFFFFFF) return fail(TS_EINVAL, "sort_period must be >= 0");
        s->sort_period = (uint32_t)value;
    } else return fail(TS_EINVAL, "unknown option '%s'", key);
    return TS_OK;
}

// ------------------------------------------------------------------ stepping

static int run_steps(ts_sim* s, uint32_t n, unsigned long long* d_digests) {
    if ((uint64_t)s->k + n >= 0x7FFFFFFFull) return fail(TS_EINVAL, "step counter would pass 2^31");
    cudaStream_t st = s->stream;
    const uint32_t R = s->sort_period;
    const uint32_t sorts = R ? (s->k + n) / R - s->k / R : 0;       // steps k with (k + 1) % R == 0
    if (s->mode == 1) {
        // one cooperative launch of `m` steps from step k0 with CTAs of `threads` threads
        auto launch = [&](uint32_t k0, uint32_t m, uint32_t cur, int threads, uint32_t variant,
                          unsigned long long* dig, uint32_t parity) -> int {
            // shared memory holds the move records of the first mr_j slots of every thread
            const int per_sm_smem = (s->smem_limit - 1024) / s->blocks_per_sm - 1024;
            uint32_t mr_j = (uint32_t)std::max(0, per_sm_smem / (16 * threads));
            const uint32_t grid = (uint32_t)(s->sms * s->blocks_per_sm);
            if (grid > kMaxCtas) return fail(TS_EINVAL, "step kernel: %u CTAs exceed the %u the sort scratch is sized for", grid, kMaxCtas);
            const uint32_t need_j = (s->L.cap + grid * threads - 1) / (grid * threads);
            mr_j = std::min(std::min(mr_j, need_j), s->smem_tiles);
            const size_t smem = (size_t)mr_j * 16 * threads;
            const void* kern = step_kernel(threads * s->blocks_per_sm, s->L.emissions != 0, s->L.ext != 0);
            int per_sm = 0;
            CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem));
            if (per_sm < s->blocks_per_sm) return fail(TS_ECUDA, "step kernel: %d CTAs of %d threads do not fit on an SM", s->blocks_per_sm, threads);
            CUDA_TRY(cudaMemsetAsync(s->ctx.barrier, 0, 4, st));
            // More warps pay once a CTA has more than one round of tiles at the small size.
            uint32_t big_above = s->adaptive_above >= 0 ? (uint32_t)s->adaptive_above : (uint32_t)s->sms * 640u;
            void* args[] = {&s->ctx, &k0, &m, &cur, (void*)&R, &mr_j, &dig, &s->profile, &variant, &big_above, &parity};
            CUDA_TRY(cudaLaunchCooperativeKernel(kern, dim3(grid), dim3(threads), args, smem, st));
            return TS_OK;
        };
        if (!s->adaptive || s->profile) {           // the phase clocks are per launch: keep it one
            int rc = launch(s->k, n, s->cur, s->threads, 2u, d_digests, 0u);
            if (rc) return rc;
            if (sorts & 1) s->cur ^= 1;
        } else {
            // Adaptive CTA size without a host round trip: the steps go out in chunks, each chunk as
            // TWO launches (640 threads, spill-free, best while a step is one warp's latency; 768
            // threads, more warps, best once CTAs hold several rounds of tiles); the device runs the
            // one the previous chunk asked for (Dyn::prefer_big) and the other returns at once.
            // Results do not depend on the launch geometry.
            // The big size: 768 threads (24 warps, 80 registers).  Measured with the 4-cell code granule, G vehicle-updates/s
            // at 704 / 736 / 768 / 800 / 832 / 896 / 960 / 1024: config 3 17.59 / 17.84 / 18.14 / 17.29 / 17.71 / 17.92 / 16.87 /
            // 17.02; the dense diagnostic 21.53 / - / 21.81 / - / 21.55 / 21.77; config 4 14.65 (704) / 15.35 (768)
            // (profiles/r02d_code_granule.md).  Until then it was 896 where the atlas fits L2.
            const int big_threads = s->adaptive_big ? s->adaptive_big : 768;
            const uint32_t chunk = s->adaptive_chunk;
            uint32_t k = s->k, cur = s->cur;
            for (uint32_t done = 0; done < n;) {
                const uint32_t m = std::min(n - done, chunk);
                unsigned long long* dig = d_digests ? d_digests + done : nullptr;
                const uint32_t parity = s->chunk_no++ & 1u;
                int rc = launch(k, m, cur, 640, 0u, dig, parity);
                if (!rc) rc = launch(k, m, cur, big_threads, 1u, dig, parity);
                if (rc) {
                    // a chunk may have run on the device without the host's step counter following:
                    // the state is no longer usable until ts_reset
                    s->sticky = ERR_LOGIC;
                    return rc;
                }
                const uint32_t srt = R ? (k + m) / R - k / R : 0;
                if (srt & 1) cur ^= 1;
                k += m; done += m;
            }
            s->cur = cur;
        }
    } else {
        const int g = s->sms * 8, gs = std::min<int>(s->sms * 8, (int)kMaxCtas);
        for (uint32_t i = 0; i < n; i++) {
            const uint32_t k = s->k + i;
            if (s->L.ext) {
                if (s->L.emissions) k_phase1<true, true><<<g, 256, 0, st>>>(s->ctx, k, s->cur);
                else k_phase1<false, true><<<g, 256, 0, st>>>(s->ctx, k, s->cur);
                k_phase2<true><<<g, 256, 0, st>>>(s->ctx, k, s->cur);
            } else {
                if (s->L.emissions) k_phase1<true, false><<<g, 256, 0, st>>>(s->ctx, k, s->cur);
                else k_phase1<false, false><<<g, 256, 0, st>>>(s->ctx, k, s->cur);
                k_phase2<false><<<g, 256, 0, st>>>(s->ctx, k, s->cur);
            }
            if (d_digests) k_digest<<<g, 256, 0, st>>>(s->ctx, s->cur, d_digests + i);
            if (R && (k + 1) % R == 0) {
                k_sort_rank<<<gs, 256, 0, st>>>(s->ctx, s->cur);
                k_sort_partial<<<gs, 256, 0, st>>>(s->ctx);
                k_sort_scan<<<gs, 256, 0, st>>>(s->ctx);
                k_sort_scatter<<<gs, 256, 0, st>>>(s->ctx, s->cur);
                s->cur ^= 1;
            }
        }
        CUDA_TRY(cudaGetLastError());
    }
    s->k += n;
    return TS_OK;
}

extern "C" int ts_step(ts_sim* s, uint32_t n) {
    if (!s) return fail(TS_EINVAL, "null sim");
    if (s->sticky) return fail(TS_EINVARIANT, "sticky device error 0x%x", s->sticky);
    if (n == 0) return TS_OK;
    return run_steps(s, n, nullptr);
}

extern "C" int ts_step_digest(ts_sim* s, uint32_t n, uint64_t* digests) {
    if (!s || !digests) return fail(TS_EINVAL, "null argument");
    if (s->sticky) return fail(TS_EINVARIANT, "sticky device error 0x%x", s->sticky);
    cudaStream_t st = s->stream;
    unsigned long long* scratch = at<unsigned long long>(s, s->L.digest);
    for (uint32_t done = 0; done < n;) {
        const uint32_t m = std::min(n - done, Layout::kDigestChunk);
        unsigned long long* d = s->out_on_device ? (unsigned long long*)digests + done : scratch;
        CUDA_TRY(cudaMemsetAsync(d, 0, (size_t)m * 8, st));
        int rc = run_steps(s, m, d);
        if (rc) return rc;
        if (!s->out_on_device) {
            CUDA_TRY(cudaMemcpyAsync(digests + done, scratch, (size_t)m * 8, cudaMemcpyDeviceToHost, st));
            CUDA_TRY(cudaStreamSynchronize(st));
        }
        done += m;
    }
    return TS_OK;
}

// ------------------------------------------------------------------ read-back

static int copy_out(ts_sim* s, void* dst, const void* src, size_t bytes) {
    if (!dst || !bytes) return TS_OK;
    CUDA_TRY(cudaMemcpyAsync(dst, src, bytes, s->out_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s->stream));
    return TS_OK;
}

static const char* describe(uint32_t err) {
    if (err & ERR_CELL_CLASH) return "atlas audit failed: two vehicles in one lane cell, or a vehicle whose cell is not marked";
    if (err & ERR_SLOTS) return "slot overflow";
    if (err & ERR_NAN) return "a vehicle's position or speed is NaN, negative or infinite";
    if (err & ERR_SPACING) return "two vehicles of one lane within one code granule (4 cells)";
    return "internal logic check failed";
}

extern "C" int ts_read_state(ts_sim* s, ts_state_out* o) {
    if (!s || !o) return fail(TS_EINVAL, "null argument");
    Layout& L = s->L;
    const size_t V = L.V;
    const bool arrays = o->status || o->edge || o->lane || o->cell || o->x || o->v || o->route_idx || o->insert_step || o->arrive_step;
    if (arrays) {
        const int g = std::max(1, std::min(1184, (int)((V + 255) / 256)));
        k_gather_slots<<<1184, 256, 0, s->stream>>>(s->ctx, s->cur);
        k_finish_state<<<g, 256, 0, s->stream>>>(s->ctx, at<uint32_t>(s, L.o_cell), at<uint32_t>(s, L.o_ridx));
        CUDA_TRY(cudaGetLastError());
    }
    int rc = 0;
    if ((rc = copy_out(s, o->status, s->ws + L.o_status, V))) return rc;
    if ((rc = copy_out(s, o->lane, s->ws + L.o_lane, V))) return rc;
    if ((rc = copy_out(s, o->edge, s->ws + L.o_edge, V * 4))) return rc;
    if ((rc = copy_out(s, o->cell, s->ws + L.o_cell, V * 4))) return rc;
    if ((rc = copy_out(s, o->x, s->ws + L.o_x, V * 4))) return rc;
    if ((rc = copy_out(s, o->v, s->ws + L.o_v, V * 4))) return rc;
    if ((rc = copy_out(s, o->route_idx, s->ws + L.o_ridx, V * 4))) return rc;
    if ((rc = copy_out(s, o->insert_step, s->ws + L.o_insert, V * 4))) return rc;
    if ((rc = copy_out(s, o->arrive_step, s->ws + L.o_arrive, V * 4))) return rc;
    unsigned long long audit[2];
    CUDA_TRY(cudaMemsetAsync(s->ctx.audit, 0, 16, s->stream));
    k_audit<<<1184, 256, 0, s->stream>>>(s->ctx, s->cur, (size_t)L.atlas_chunks * 4);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaMemcpyAsync(audit, s->ctx.audit, 16, cudaMemcpyDeviceToHost, s->stream));
    Dyn d;
    CUDA_TRY(cudaMemcpyAsync(&d, s->ws + L.dyn, sizeof d, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    if (audit[1] || audit[0] != (unsigned long long)(d.n_departed - d.n_arrived)) d.error |= ERR_CELL_CLASH;
    o->step = s->k; o->n_pending = L.V - d.n_departed; o->n_active = d.n_departed - d.n_arrived; o->n_arrived = d.n_arrived;
    o->vehicle_updates = d.updates;
    if (d.error) { s->sticky = d.error; return fail(TS_EINVARIANT, "device invariant violated (flags 0x%x): %s", d.error, describe(d.error)); }
    return TS_OK;
}

extern "C" int ts_read_profile(ts_sim* s, uint64_t out[8]) {
    if (!s || !out) return fail(TS_EINVAL, "null argument");
    Dyn d;
    CUDA_TRY(cudaMemcpyAsync(&d, s->ws + s->L.dyn, sizeof d, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    for (int b = 0; b < 8; b++) out[b] = d.prof[b];
    return TS_OK;
}

// totals of the vehicles still driving: slot-ordered -> id-ordered (arrived ones are there already)
__global__ void k_gather_emissions(const __grid_constant__ Ctx c, uint32_t cur) {
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nthreads = gridDim.x * blockDim.x;
    const uint32_t n_slots = min(c.dyn->slot_alloc, c.cap_slots);
    const Slots& S = c.s[cur];
    for (uint32_t s = tid; s < n_slots; s += nthreads)
        if (S.A[s].w & ALIVE) c.emis[S.B[s].z] = S.D[s];
}

// id-ordered { CO, fuel } pairs -> two plain arrays (staged in ts_read_state's scratch)
__global__ void k_split_emissions(const float2* __restrict__ emis, uint32_t V, float* co, float* fuel) {
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < V; i += gridDim.x * blockDim.x) {
        const float2 e = emis[i];
        co[i] = e.x; fuel[i] = e.y;
    }
}

extern "C" int ts_read_emissions(ts_sim* s, float* co_g, float* fuel_ml) {
    if (!s) return fail(TS_EINVAL, "null sim");
    Layout& L = s->L;
    if (!L.emissions) return fail(TS_EINVAL, "the simulation was created with ts_params.emissions == 0");
    const size_t V = L.V;
    if (V) {
        k_gather_emissions<<<1184, 256, 0, s->stream>>>(s->ctx, s->cur);
        k_split_emissions<<<(unsigned)std::min<size_t>(1184, (V + 255) / 256), 256, 0, s->stream>>>(
            s->ctx.emis, L.V, at<float>(s, L.o_cell), at<float>(s, L.o_ridx));
        CUDA_TRY(cudaGetLastError());
    }
    int rc = 0;
    if ((rc = copy_out(s, co_g, s->ws + L.o_cell, V * 4))) return rc;
    if ((rc = copy_out(s, fuel_ml, s->ws + L.o_ridx, V * 4))) return rc;
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    return TS_OK;
}

extern "C" int ts_read_edge_stats(ts_sim* s, ts_edge_stats_out* o, int reset) {
    if (!s || !o) return fail(TS_EINVAL, "null argument");
    Layout& L = s->L;
    const size_t E = L.E;
    int rc = 0;
    if ((rc = copy_out(s, o->entered, s->ws + L.st_entered, E * 4))) return rc;
    if ((rc = copy_out(s, o->exited, s->ws + L.st_exited, E * 4))) return rc;
    if ((rc = copy_out(s, o->exit_steps_sum, s->ws + L.st_exit_steps, E * 8))) return rc;
    if ((rc = copy_out(s, o->sample_count_sum, s->ws + L.st_samp_cnt, E * 4))) return rc;
    if ((rc = copy_out(s, o->sample_speedcode_sum, s->ws + L.st_samp_code, E * 8))) return rc;
    Dyn d;
    CUDA_TRY(cudaMemcpyAsync(&d, s->ws + L.dyn, sizeof d, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    o->n_samples = d.n_samples;
    if (reset) {
        CUDA_TRY(cudaMemsetAsync(s->ws + L.st_entered, 0, L.emis - L.st_entered, s->stream));
        CUDA_TRY(cudaMemsetAsync(s->ws + L.dyn + offsetof(Dyn, n_samples), 0, 4, s->stream));
    }
    return TS_OK;
}

// "We defined utilization as the number of vehicles at the sampling time divided by the
// maximum number of vehicles that can fit on the edge.  This capacity is computed as the length of the
// edge times the number of lines divided by the average length of a vehicle plus the lead gap" -- and the
// per-edge speed of PAPER.md:437, both averaged over the samples taken since the last reset.
__global__ void k_utilisation(const __grid_constant__ Ctx c, float* util, float* speed) {
    const uint32_t n_samples = c.dyn->n_samples;
    for (uint32_t e = blockIdx.x * blockDim.x + threadIdx.x; e < c.E; e += gridDim.x * blockDim.x) {
        const EdgeRec E = c.edges[e];
        const float cap = ((float)E.len * (float)edge_lanes(E)) / (c.p.len + c.p.s0);
        const uint32_t cnt = c.st_samp_cnt[e];
        util[e] = n_samples ? ((float)cnt / (float)n_samples) / cap : 0.0f;
        speed[e] = cnt ? ((float)c.st_samp_code[e] * 0.25f) / (float)cnt : 0.0f;
    }
}

extern "C" int ts_read_utilisation(ts_sim* s, float* utilisation, float* mean_speed) {
    if (!s) return fail(TS_EINVAL, "null sim");
    Layout& L = s->L;
    k_utilisation<<<std::max(1u, std::min(1184u, (L.E + 255) / 256)), 256, 0, s->stream>>>(s->ctx, at<float>(s, L.o_cell), at<float>(s, L.o_ridx));
    CUDA_TRY(cudaGetLastError());
    int rc = 0;
    if ((rc = copy_out(s, utilisation, s->ws + L.o_cell, (size_t)L.E * 4))) return rc;
    if ((rc = copy_out(s, mean_speed, s->ws + L.o_ridx, (size_t)L.E * 4))) return rc;
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    return TS_OK;
}

// ------------------------------------------------------------------ re-routing

extern "C" int ts_reroute(ts_sim* s, const uint32_t* w_free, const uint8_t* mask, ts_reroute_out* out) {
    if (!s || !w_free) return fail(TS_EINVAL, "null argument");
    Layout& L = s->L;
    if (!L.Rcap) return fail(TS_EINVAL, "the simulation was created with ts_params.route_capacity == 0");
    if (s->sticky) return fail(TS_EINVARIANT, "sticky device error 0x%x", s->sticky);
    const uint32_t V = L.V, E = L.E;
    cudaStream_t st = s->stream;
    RrCtx& r = s->rr;
    // route tables: the one in use and the one to fill
    uint32_t* tab[2] = {at<uint32_t>(s, L.route_edges), at<uint32_t>(s, L.rr_routes2)};
    r.old_routes = tab[s->route_cur]; r.new_routes = tab[s->route_cur ^ 1];
    r.old_begin = at<uint32_t>(s, L.route_begin); r.old_end = at<uint32_t>(s, L.rr_end);
    for (uint32_t e = 0; e < E; e++)
        if (w_free[e] < 1 || w_free[e] > kRrWMax) return fail(TS_EINVAL, "w_free[%u] = %u not in 1..2^20", e, w_free[e]);
    CUDA_TRY(cudaMemcpyAsync(s->ws + L.rr_wfree, w_free, (size_t)E * 4, cudaMemcpyHostToDevice, st));
    if (mask) CUDA_TRY(cudaMemcpyAsync(s->ws + L.rr_mask, mask, V, cudaMemcpyHostToDevice, st));
    else CUDA_TRY(cudaMemsetAsync(s->ws + L.rr_mask, 1, V, st));
    CUDA_TRY(cudaMemsetAsync(r.error, 0, 4, st));
    // the trees wanted: origins of the vehicles asked to re-route (R39)
    std::vector<uint8_t> want(L.n_src, 0);
    std::vector<uint32_t> todo;
    uint32_t n_masked = 0;
    for (uint32_t i = 0; i < V; i++)
        if (!mask || mask[i]) { n_masked++; if (!want[s->src_idx_h[i]]) { want[s->src_idx_h[i]] = 1; todo.push_back(s->src_idx_h[i]); } }
    std::sort(todo.begin(), todo.end());
    CUDA_TRY(cudaMemcpyAsync(s->ws + L.rr_todo, todo.data(), todo.size() * 4, cudaMemcpyHostToDevice, st));
    cudaEvent_t ev[3];
    for (auto& e : ev) CUDA_TRY(cudaEventCreate(&e));
    k_rr_weights<<<std::max(1u, std::min(1184u, (E + 255) / 256)), 256, 0, st>>>(r);
    CUDA_TRY(cudaEventRecord(ev[0], st));
    if (!todo.empty()) {
        k_rr_pack<<<std::max(1u, std::min(1184u, (E + 255) / 256)), 256, 0, st>>>(r);
        k_rr_sssp<<<std::min<uint32_t>(kRrCtas, (uint32_t)todo.size()), kRrThreads, 0, st>>>(r, at<uint32_t>(s, L.rr_todo), (uint32_t)todo.size());
    }
    CUDA_TRY(cudaEventRecord(ev[1], st));
    const uint32_t vb = std::max(1u, std::min(1184u, (V + 255) / 256));
    k_rr_len<<<vb, 256, 0, st>>>(r);
    CUDA_TRY(cudaMemsetAsync(r.new_len + V, 0, 4, st));
    const uint32_t n_scan = V + 1, per = kScanBlock * kScanItems, nb = (n_scan + per - 1) / per;
    k_rr_scan1<<<nb, kScanBlock, 0, st>>>(r.new_len, r.new_off, r.block_sum, n_scan);
    k_rr_scan2<<<1, 32, 0, st>>>(r.block_sum, nb);
    k_rr_scan3<<<nb, kScanBlock, 0, st>>>(r.new_off, r.block_sum, n_scan);
    CUDA_TRY(cudaGetLastError());
    // the total decides whether the new routes fit (lengths sum below 2^32: every route has at most N edges
    // and the scan is checked against the capacity before anything is written)
    uint32_t total = 0, err = 0;
    std::vector<uint32_t> new_len(V), new_off((size_t)V + 1);
    CUDA_TRY(cudaMemcpyAsync(new_len.data(), r.new_len, (size_t)V * 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(new_off.data(), r.new_off, ((size_t)V + 1) * 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(&err, r.error, 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (err) return fail(TS_EINVAL, "re-routing: a path cost passed 2^32 weight units");
    uint64_t sum = 0;
    for (uint32_t i = 0; i < V; i++) sum += new_len[i];
    total = new_off[V];
    if (sum > L.Rcap || sum != total) return fail(TS_ENOMEM, "re-routing: the new routes need %llu entries, route_capacity is %llu", (unsigned long long)sum, (unsigned long long)L.Rcap);
    k_rr_write<<<vb, 256, 0, st>>>(r);
    k_rr_first2<<<vb, 256, 0, st>>>(r);
    CUDA_TRY(cudaEventRecord(ev[2], st));
    CUDA_TRY(cudaGetLastError());
    // the departure-queue index follows the new first edges (host: a counting sort and one record per vehicle)
    std::vector<uint32_t> first2(2 * (size_t)V), first(V), second(V), rend(V);
    CUDA_TRY(cudaMemcpyAsync(first2.data(), r.first2, (size_t)V * 8, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    for (uint32_t i = 0; i < V; i++) { first[i] = first2[2 * (size_t)i]; second[i] = first2[2 * (size_t)i + 1]; rend[i] = new_off[i] + new_len[i]; }
    DepRecBuf dep_rec;
    std::vector<uint4> queue_rec;
    build_queues(V, E, s->edges_h, first.data(), second.data(), new_off.data(), rend.data(), s->dep_step_h.data(),
                 s->v0m_bits_h.data(), s->mand_bits_h.data(), s->type_h.data(), dep_rec, queue_rec);
    if (queue_rec.size() > std::max(L.Q, L.Qcap)) return fail(TS_ENOMEM, "re-routing: %zu departure queues, room for %u", queue_rec.size(), std::max(L.Q, L.Qcap));
    CUDA_TRY(cudaMemcpyAsync(s->ws + L.queue_rec, queue_rec.data(), queue_rec.size() * 16, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(s->ws + L.dep_rec, dep_rec.data(), (size_t)V * 32, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(s->ws + L.route_begin, r.new_off, (size_t)V * 4, cudaMemcpyDeviceToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(s->ws + L.rr_end, rend.data(), (size_t)V * 4, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    s->route_cur ^= 1;
    s->ctx.route_edges = tab[s->route_cur];
    s->ctx.n_queues = (uint32_t)queue_rec.size();
    if (out) {
        float ms_sssp = 0, ms_all = 0;
        cudaEventElapsedTime(&ms_sssp, ev[0], ev[1]);
        cudaEventElapsedTime(&ms_all, ev[0], ev[2]);
        out->n_rerouted = n_masked; out->n_trees = (uint32_t)todo.size(); out->route_entries = sum;
        out->sssp_ms = ms_sssp; out->device_ms = ms_all;
        if (out->w) CUDA_TRY(cudaMemcpyAsync(out->w, r.w, (size_t)E * 4, s->out_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, st));
    }
    for (auto& e : ev) cudaEventDestroy(e);
    return ts_reset(s);       // new demand: back to step 0, statistics cleared
}

extern "C" int ts_read_routes(ts_sim* s, uint64_t* route_off, uint32_t* route_edges, uint64_t* n_entries) {
    if (!s) return fail(TS_EINVAL, "null sim");
    Layout& L = s->L;
    const uint32_t V = L.V;
    cudaStream_t st = s->stream;
    std::vector<uint32_t> b(V), e(V);
    CUDA_TRY(cudaMemcpyAsync(b.data(), s->ws + L.route_begin, (size_t)V * 4, cudaMemcpyDeviceToHost, st));
    if (L.Rcap) CUDA_TRY(cudaMemcpyAsync(e.data(), s->ws + L.rr_end, (size_t)V * 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    const uint64_t total = L.Rcap ? (V ? e[V - 1] : 0) : L.R;      // routes are stored back to back in id order
    if (n_entries) *n_entries = total;
    if (route_off) {
        if (s->out_on_device) return fail(TS_EINVAL, "ts_read_routes fills host arrays");
        for (uint32_t i = 0; i < V; i++) route_off[i] = b[i];
        route_off[V] = total;
    }
    if (route_edges) {
        CUDA_TRY(cudaMemcpyAsync(route_edges, s->ctx.route_edges, total * 4, cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
    }
    return TS_OK;
}

// ------------------------------------------------------------------ static user equilibrium

struct SueLayout {
    size_t total = 0;
    size_t out_off, out_edge, efrom, eto, t0, cap, x, t, w, y, part, od_o, od_d, od_t, od_s, src, todo, pred, lab, fa, fb, stamp, err, adjw;
    uint32_t n_src = 0;
    size_t take(size_t bytes) { size_t off = total; total += (bytes + 255) & ~(size_t)255; return off; }
    void plan(uint32_t N, uint32_t E, uint32_t n_od) {
        out_off = take(((size_t)N + 1) * 4); out_edge = take((size_t)E * 4); efrom = take((size_t)E * 4); eto = take((size_t)E * 4);
        t0 = take((size_t)E * 8); cap = take((size_t)E * 8); x = take((size_t)E * 8); t = take((size_t)E * 8);
        w = take((size_t)E * 4); y = take((size_t)E * 8); part = take((size_t)kSueBlocks * 2 * 8);
        od_o = take((size_t)n_od * 4); od_d = take((size_t)n_od * 4); od_t = take((size_t)n_od * 4); od_s = take((size_t)n_od * 4);
        src = take((size_t)n_src * 4); todo = take((size_t)n_src * 4); pred = take((size_t)n_src * N * 4);
        lab = take((size_t)kRrCtas * N * 8); fa = take((size_t)kRrCtas * N * 8); fb = take((size_t)kRrCtas * N * 8);
        stamp = take((size_t)kRrCtas * N * 4); err = take(4);
        adjw = take(((size_t)E + 4) * 16);
    }
};

static int sue_plan(const ts_sue_problem* p, SueLayout& L, std::vector<uint32_t>* src_nodes, std::vector<uint32_t>* od_src) {
    if (!p || !p->edge_from || !p->edge_to || !p->t0 || !p->cap || (p->n_od && (!p->od_origin || !p->od_dest || !p->od_trips)))
        return fail(TS_EINVAL, "null argument");
    if (p->n_nodes == 0 || p->n_edges == 0) return fail(TS_EINVAL, "empty network");
    if (p->n_edges >= 0x80000000u) return fail(TS_EINVAL, "more than 2^31 edges");
    if (!(p->alpha >= 0) || !(p->weight_scale > 0) || p->bisections > 64) return fail(TS_EINVAL, "alpha >= 0, weight_scale > 0, bisections <= 64");
    for (uint32_t e = 0; e < p->n_edges; e++) {
        if (p->edge_from[e] >= p->n_nodes || p->edge_to[e] >= p->n_nodes) return fail(TS_EINVAL, "edge %u: endpoint out of range", e);
        if (!(p->t0[e] > 0) || !(p->cap[e] > 0)) return fail(TS_EINVAL, "edge %u: t0 and cap must be > 0", e);
    }
    std::vector<uint32_t> idx_of(p->n_nodes, NONE32), srcs;
    if (od_src) od_src->resize(p->n_od);
    for (uint32_t q = 0; q < p->n_od; q++) {
        if (p->od_origin[q] >= p->n_nodes || p->od_dest[q] >= p->n_nodes) return fail(TS_EINVAL, "OD pair %u: node out of range", q);
        const uint32_t o = p->od_origin[q];
        if (idx_of[o] == NONE32) { idx_of[o] = (uint32_t)srcs.size(); srcs.push_back(o); }
        if (od_src) (*od_src)[q] = idx_of[o];
    }
    L.n_src = (uint32_t)srcs.size();
    L.plan(p->n_nodes, p->n_edges, p->n_od);
    if (src_nodes) *src_nodes = srcs;
    return TS_OK;
}

extern "C" int ts_sue_workspace(const ts_sue_problem* p, size_t* bytes) {
    if (!bytes) return fail(TS_EINVAL, "bytes is null");
    SueLayout L;
    int rc = sue_plan(p, L, nullptr, nullptr);
    if (rc) return rc;
    *bytes = L.total;
    return TS_OK;
}

extern "C" int ts_sue_solve(const ts_sue_problem* p, const ts_device* dev, ts_sue_out* out) {
    if (!dev || !out) return fail(TS_EINVAL, "null argument");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(TS_ECUDA, "no CUDA device: this library has no CPU fallback");
    SueLayout L;
    std::vector<uint32_t> srcs, od_src;
    int rc = sue_plan(p, L, &srcs, &od_src);
    if (rc) return rc;
    if (!dev->workspace || ((uintptr_t)dev->workspace & 255)) return fail(TS_EINVAL, "workspace must be a 256-byte aligned device pointer");
    if (dev->bytes < L.total) return fail(TS_ENOMEM, "workspace too small: %zu < %zu bytes", dev->bytes, L.total);
    uint8_t* ws = (uint8_t*)dev->workspace;
    cudaStream_t st = (cudaStream_t)dev->cuda_stream;
    const uint32_t N = p->n_nodes, E = p->n_edges, n_od = p->n_od;
    std::vector<uint32_t> out_off((size_t)N + 1, 0), out_edge(E), todo(L.n_src);
    for (uint32_t e = 0; e < E; e++) out_off[p->edge_from[e] + 1]++;
    for (uint32_t h = 0; h < N; h++) out_off[h + 1] += out_off[h];
    { std::vector<uint32_t> fill(out_off.begin(), out_off.end() - 1);
      for (uint32_t e = 0; e < E; e++) out_edge[fill[p->edge_from[e]]++] = e; }
    for (uint32_t i = 0; i < L.n_src; i++) todo[i] = i;
    auto up = [&](size_t off, const void* src, size_t bytes) { return bytes ? cudaMemcpyAsync(ws + off, src, bytes, cudaMemcpyHostToDevice, st) : cudaSuccess; };
    CUDA_TRY(up(L.out_off, out_off.data(), ((size_t)N + 1) * 4)); CUDA_TRY(up(L.out_edge, out_edge.data(), (size_t)E * 4));
    CUDA_TRY(up(L.efrom, p->edge_from, (size_t)E * 4)); CUDA_TRY(up(L.eto, p->edge_to, (size_t)E * 4));
    CUDA_TRY(up(L.t0, p->t0, (size_t)E * 8)); CUDA_TRY(up(L.cap, p->cap, (size_t)E * 8));
    CUDA_TRY(up(L.od_o, p->od_origin, (size_t)n_od * 4)); CUDA_TRY(up(L.od_d, p->od_dest, (size_t)n_od * 4));
    CUDA_TRY(up(L.od_t, p->od_trips, (size_t)n_od * 4)); CUDA_TRY(up(L.od_s, od_src.data(), (size_t)n_od * 4));
    CUDA_TRY(up(L.src, srcs.data(), (size_t)L.n_src * 4)); CUDA_TRY(up(L.todo, todo.data(), (size_t)L.n_src * 4));
    CUDA_TRY(cudaMemsetAsync(ws + L.err, 0, 4, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    auto dp = [&](size_t off) { return reinterpret_cast<double*>(ws + off); };
    auto up32 = [&](size_t off) { return reinterpret_cast<uint32_t*>(ws + off); };
    RrCtx r;
    memset(&r, 0, sizeof r);
    r.N = N; r.E = E; r.n_src = L.n_src;
    r.out_off = up32(L.out_off); r.out_edge = up32(L.out_edge); r.edge_from = up32(L.efrom); r.edge_to = up32(L.eto);
    r.w = up32(L.w); r.src_node = up32(L.src); r.pred = up32(L.pred);
    r.lab = reinterpret_cast<unsigned long long*>(ws + L.lab); r.fa = reinterpret_cast<uint2*>(ws + L.fa); r.fb = reinterpret_cast<uint2*>(ws + L.fb); r.stamp = up32(L.stamp);
    r.error = up32(L.err); r.adjw = reinterpret_cast<uint4*>(ws + L.adjw);
    unsigned long long* y = reinterpret_cast<unsigned long long*>(ws + L.y);
    const uint32_t eb = std::max(1u, std::min(1184u, (E + 255) / 256)), ob = std::max(1u, std::min(1184u, (n_od + 255) / 256));
    cudaEvent_t ev0, ev1, t0e, t1e;
    CUDA_TRY(cudaEventCreate(&ev0)); CUDA_TRY(cudaEventCreate(&ev1)); CUDA_TRY(cudaEventCreate(&t0e)); CUDA_TRY(cudaEventCreate(&t1e));
    float sssp_ms = 0;
    double part[2 * kSueBlocks];
    // one all-or-nothing assignment on the times of flow x (nullptr: free flow) into y
    auto assign = [&](const double* x) -> int {
        k_sue_times<<<eb, 256, 0, st>>>(E, dp(L.t0), dp(L.cap), x, p->alpha, p->weight_scale, dp(L.t), r.w);
        CUDA_TRY(cudaEventRecord(t0e, st));
        if (L.n_src) {
            k_rr_pack<<<eb, 256, 0, st>>>(r);
            k_rr_sssp<<<std::min<uint32_t>(kRrCtas, L.n_src), kRrThreads, 0, st>>>(r, up32(L.todo), L.n_src);
        }
        CUDA_TRY(cudaEventRecord(t1e, st));
        CUDA_TRY(cudaMemsetAsync(y, 0, (size_t)E * 8, st));
        if (n_od) k_sue_aon<<<ob, 256, 0, st>>>(n_od, up32(L.od_o), up32(L.od_d), up32(L.od_t), up32(L.od_s), r.pred, N, r.edge_from, y);
        CUDA_TRY(cudaGetLastError());
        CUDA_TRY(cudaEventSynchronize(t1e));
        float ms = 0; cudaEventElapsedTime(&ms, t0e, t1e); sssp_ms += ms;
        return TS_OK;
    };
    // block sums added up in block order on the host: the same sum whatever the scheduling
    auto reduce = [&](int mode, double a, double& s0, double& s1) -> int {
        k_sue_reduce<<<kSueBlocks, kSueThreads, 0, st>>>(mode, E, dp(L.t0), dp(L.cap), dp(L.x), y, a, p->alpha, dp(L.part));
        CUDA_TRY(cudaMemcpyAsync(part, ws + L.part, sizeof part, cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
        s0 = s1 = 0.0;
        for (uint32_t b = 0; b < kSueBlocks; b++) { s0 += part[b]; s1 += part[kSueBlocks + b]; }
        return TS_OK;
    };
    CUDA_TRY(cudaEventRecord(ev0, st));
    double s0, s1;
    if ((rc = assign(nullptr))) return rc;                                     // step 1: x_0
    k_sue_update<<<eb, 256, 0, st>>>(E, dp(L.x), y, 0.0, 1);
    if ((rc = reduce(1, 0.0, s0, s1))) return rc;
    if (out->objective) out->objective[0] = s0;
    for (uint32_t k = 0; k < p->iterations; k++) {
        if ((rc = assign(dp(L.x)))) return rc;                                 // step 2: y_k
        if ((rc = reduce(2, 0.0, s0, s1))) return rc;
        if (out->gap) out->gap[k] = (s0 - s1) / s0;
        double a, g1, g0;                                                      // step 3: step length
        if ((rc = reduce(0, 1.0, g1, s1))) return rc;
        if (g1 <= 0.0) a = 1.0;
        else {
            if ((rc = reduce(0, 0.0, g0, s1))) return rc;
            if (g0 >= 0.0) a = 0.0;
            else {
                double lo = 0.0, hi = 1.0;
                for (uint32_t b = 0; b < p->bisections; b++) {
                    const double mid = 0.5 * (lo + hi);
                    double g;
                    if ((rc = reduce(0, mid, g, s1))) return rc;
                    if (g > 0.0) hi = mid; else lo = mid;
                }
                a = 0.5 * (lo + hi);
            }
        }
        k_sue_update<<<eb, 256, 0, st>>>(E, dp(L.x), y, a, 0);                 // step 4
        if (out->step) out->step[k] = a;
        if ((rc = reduce(1, 0.0, s0, s1))) return rc;
        if (out->objective) out->objective[k + 1] = s0;
    }
    k_sue_times<<<eb, 256, 0, st>>>(E, dp(L.t0), dp(L.cap), dp(L.x), p->alpha, p->weight_scale, dp(L.t), r.w);
    CUDA_TRY(cudaEventRecord(ev1, st));
    const cudaMemcpyKind kind = dev->out_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    if (out->flow) CUDA_TRY(cudaMemcpyAsync(out->flow, ws + L.x, (size_t)E * 8, kind, st));
    if (out->time) CUDA_TRY(cudaMemcpyAsync(out->time, ws + L.t, (size_t)E * 8, kind, st));
    uint32_t err = 0;
    CUDA_TRY(cudaMemcpyAsync(&err, ws + L.err, 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    float ms = 0; cudaEventElapsedTime(&ms, ev0, ev1);
    out->device_ms = ms; out->sssp_ms = sssp_ms; out->n_trees = L.n_src * (p->iterations + 1);
    cudaEventDestroy(ev0); cudaEventDestroy(ev1); cudaEventDestroy(t0e); cudaEventDestroy(t1e);
    if (err) return fail(TS_EINVAL, "a path cost passed 2^32 weight units: lower weight_scale");
    return TS_OK;
}

// ------------------------------------------------------------------ shortest-path trees without any allocation
//
// ts_sssp_static: the tree kernel of ts_reroute / ts_sue_solve for callers that cannot allocate (CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc).  Its scratch -- per tree in flight a 64-bit
// label, two frontier words and a stamp per node -- lives in ONE file-scope device array of a fixed size, which
// every GPU that loads this library holds until the process exits.  Nothing here calls cudaMalloc, cudaFree, an
// allocating library routine or the host allocator; the call only enqueues one kernel on the caller's stream.
//
// The array keeps the last call's contents.  Nothing needs clearing between calls: the kernel initialises the
// labels and stamps of a tree before it grows it, and never reads a frontier slot it did not write.  All calls on
// one GPU SHARE the array: two calls that overlap on the GPU (different streams, no dependency) race.
constexpr size_t kStaticScratchBytes = (size_t)20 << 20;          // 20 MiB per GPU
constexpr uint32_t kStaticMaxNodes = 65536;                        // 20 bytes of scratch per node and tree: 16 trees in flight
constexpr uint32_t kStaticBytesPerNode = 20;
static __device__ __align__(256) unsigned char g_sssp_scratch[kStaticScratchBytes];

// Same relaxation rule as k_rr_sssp (ts_reroute.cuh; from the caller's CSR arrays here, from packed records there: the
// labels at the end are the same minimum), trees numbered 0..n_src-1 in the caller's source order;
// `scratch` is the device address of g_sssp_scratch (device code could name the array directly, the host cannot).
__global__ void __launch_bounds__(kRrThreads) k_sssp_static(unsigned char* scratch, uint32_t N, const uint32_t* __restrict__ out_off,
                                                            const uint32_t* __restrict__ out_edge, const uint32_t* __restrict__ edge_to,
                                                            const uint32_t* __restrict__ w, const uint32_t* __restrict__ sources,
                                                            uint32_t n_src, uint32_t* __restrict__ pred, uint32_t* error) {
    __shared__ uint32_t sh_next;
    const uint32_t t = threadIdx.x, T = blockDim.x, n_cta = gridDim.x;
    unsigned long long* lab = reinterpret_cast<unsigned long long*>(scratch) + (size_t)blockIdx.x * N;
    uint32_t* words = reinterpret_cast<uint32_t*>(scratch + (size_t)n_cta * N * 8);
    uint32_t* fa = words + ((size_t)0 * n_cta + blockIdx.x) * N;
    uint32_t* fb = words + ((size_t)1 * n_cta + blockIdx.x) * N;
    uint32_t* stamp = words + ((size_t)2 * n_cta + blockIdx.x) * N;
    for (uint32_t si = blockIdx.x; si < n_src; si += n_cta) {
        const uint32_t s = sources[si];
        for (uint32_t v = t; v < N; v += T) { lab[v] = ~0ull; stamp[v] = 0u; }
        __syncthreads();
        if (t == 0) { lab[s] = (unsigned long long)kRrNone; fa[0] = s; sh_next = 0; }
        __syncthreads();
        uint32_t n_f = 1, epoch = 0;
        while (n_f) {
            epoch++;
            for (uint32_t i = t; i < n_f; i += T) {
                const uint32_t u = __ldcg(fa + i);
                const unsigned long long du = __ldcg(lab + u) >> 32;
                const uint32_t j1 = out_off[u + 1];
                // four outbound edges at a time, every load of a stage issued before any is consumed (k_rr_sssp
                // does the same from packed records, which this call has no scratch for)
                for (uint32_t j = out_off[u]; j < j1; j += 4) {
                    uint32_t e[4], v[4], we[4], seen[4];
                    unsigned long long cand[4], old[4];
                    bool go[4];
#pragma unroll
                    for (int q = 0; q < 4; q++) { go[q] = j + q < j1; e[q] = go[q] ? out_edge[j + q] : 0u; }
#pragma unroll
                    for (int q = 0; q < 4; q++) if (go[q]) { v[q] = edge_to[e[q]]; we[q] = w[e[q]]; }
#pragma unroll
                    for (int q = 0; q < 4; q++) if (go[q]) {
                        const unsigned long long nd = du + we[q];
                        if (nd >= 0xFFFFFFFFull) { if (error) *error = 1u; go[q] = false; }
                        cand[q] = (nd << 32) | e[q];
                    }
#pragma unroll
                    for (int q = 0; q < 4; q++) if (go[q]) old[q] = atomicMin(lab + v[q], cand[q]);
#pragma unroll
                    for (int q = 0; q < 4; q++) {
                        go[q] = go[q] && cand[q] < old[q] && (cand[q] >> 32) < (old[q] >> 32);
                        if (go[q]) seen[q] = atomicExch(stamp + v[q], epoch);
                    }
#pragma unroll
                    for (int q = 0; q < 4; q++) if (go[q] && seen[q] != epoch) fb[atomicAdd(&sh_next, 1u)] = v[q];
                }
            }
            __syncthreads();
            n_f = sh_next;
            __syncthreads();
            if (t == 0) sh_next = 0;
            uint32_t* tmp = fa; fa = fb; fb = tmp;
            __threadfence_block();
            __syncthreads();
        }
        uint32_t* row = pred + (size_t)si * N;
        for (uint32_t v = t; v < N; v += T) row[v] = (uint32_t)__ldcg(lab + v);
        __syncthreads();
    }
}

// Device address of g_sssp_scratch, resolved once per device with that device current.  In host code the
// array's NAME is a host-side stand-in, not a device address: only cudaGetSymbolAddress gives the address.
constexpr int kStaticMaxDevices = 64;
static std::atomic<unsigned char*> g_sssp_scratch_ptr[kStaticMaxDevices];

extern "C" uint32_t ts_sssp_static_max_nodes(void) { return kStaticMaxNodes; }

extern "C" int ts_sssp_static(uint32_t n_nodes, uint32_t n_edges, const uint32_t* d_out_off, const uint32_t* d_out_edge,
                              const uint32_t* d_edge_to, const uint32_t* d_w, const uint32_t* d_sources,
                              uint32_t n_sources, uint32_t* d_pred, uint32_t* d_error, void* cuda_stream) {
    if (n_nodes == 0 || n_edges == 0) return fail(TS_EINVAL, "empty graph");
    if (n_nodes > kStaticMaxNodes)
        return fail(TS_EINVAL, "ts_sssp_static: %u nodes exceed the %u its static scratch of %zu MiB is sized for "
                               "(use ts_reroute / ts_sue_solve with a caller-owned workspace)", n_nodes, kStaticMaxNodes,
                    kStaticScratchBytes >> 20);
    if (!d_out_off || !d_out_edge || !d_edge_to || !d_w || (n_sources && (!d_sources || !d_pred)))
        return fail(TS_EINVAL, "null argument");
    if (n_sources == 0) return TS_OK;
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(TS_EINVAL, "device ordinal %d beyond %d", dev, kStaticMaxDevices);
    unsigned char* scratch = g_sssp_scratch_ptr[dev].load(std::memory_order_acquire);
    if (!scratch) {                                  // set-up, once per device, with that device current
        void* p = nullptr;
        CUDA_TRY(cudaGetSymbolAddress(&p, g_sssp_scratch));
        scratch = static_cast<unsigned char*>(p);
        g_sssp_scratch_ptr[dev].store(scratch, std::memory_order_release);
    }
    const uint64_t per_tree = (uint64_t)n_nodes * kStaticBytesPerNode;
    const uint32_t ctas = (uint32_t)std::min<uint64_t>({(uint64_t)kRrCtas, (uint64_t)n_sources, kStaticScratchBytes / per_tree});
    k_sssp_static<<<ctas, kRrThreads, 0, (cudaStream_t)cuda_stream>>>(scratch, n_nodes, d_out_off, d_out_edge, d_edge_to, d_w,
                                                                       d_sources, n_sources, d_pred, d_error);
    CUDA_TRY(cudaGetLastError());
    return TS_OK;
}

// ------------------------------------------------------------------ checkpoint / resume
//
// The caller owns the whole workspace, so a checkpoint is a copy of it (without the shortest-path scratch of
// ts_reroute, which holds nothing between calls) behind a small header with the host-side counters.  Restoring
// needs a simulation created from the SAME inputs (same layout); the header is checked for that.
struct CheckpointHeader {
    uint64_t magic, ws_bytes, total;
    uint32_t V, E, N, k, cur, chunk_no, route_cur, n_queues, sticky, pad;
};
static constexpr uint64_t kCheckpointMagic = 0x31544B4350435354ull;   // "TSCPCKT1"

static size_t checkpoint_ws_bytes(const ts_sim* s) { return s->L.Rcap ? s->L.rr_pred : s->L.total; }

extern "C" int ts_checkpoint_size(ts_sim* s, size_t* bytes) {
    if (!s || !bytes) return fail(TS_EINVAL, "null argument");
    *bytes = sizeof(CheckpointHeader) + checkpoint_ws_bytes(s);
    return TS_OK;
}

extern "C" int ts_checkpoint(ts_sim* s, void* host_buf) {
    if (!s || !host_buf) return fail(TS_EINVAL, "null argument");
    if (s->sticky) return fail(TS_EINVARIANT, "sticky device error 0x%x", s->sticky);
    CheckpointHeader h;
    memset(&h, 0, sizeof h);
    h.magic = kCheckpointMagic; h.ws_bytes = checkpoint_ws_bytes(s); h.total = s->L.total;
    h.V = s->L.V; h.E = s->L.E; h.N = s->L.N; h.k = s->k; h.cur = s->cur; h.chunk_no = s->chunk_no;
    h.route_cur = s->route_cur; h.n_queues = s->ctx.n_queues; h.sticky = s->sticky;
    memcpy(host_buf, &h, sizeof h);
    CUDA_TRY(cudaMemcpyAsync((uint8_t*)host_buf + sizeof h, s->ws, h.ws_bytes, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    return TS_OK;
}

extern "C" int ts_restore(ts_sim* s, const void* host_buf) {
    if (!s || !host_buf) return fail(TS_EINVAL, "null argument");
    CheckpointHeader h;
    memcpy(&h, host_buf, sizeof h);
    if (h.magic != kCheckpointMagic) return fail(TS_EINVAL, "not a checkpoint of this library");
    if (h.total != s->L.total || h.ws_bytes != checkpoint_ws_bytes(s) || h.V != s->L.V || h.E != s->L.E || h.N != s->L.N)
        return fail(TS_EINVAL, "the checkpoint was taken from a simulation with other inputs (workspace layout differs)");
    CUDA_TRY(cudaMemcpyAsync(s->ws, (const uint8_t*)host_buf + sizeof h, h.ws_bytes, cudaMemcpyHostToDevice, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    s->k = h.k; s->cur = h.cur; s->chunk_no = h.chunk_no; s->sticky = h.sticky;
    s->route_cur = h.route_cur; s->ctx.n_queues = h.n_queues;
    if (s->L.Rcap) s->ctx.route_edges = at<uint32_t>(s, h.route_cur ? s->L.rr_routes2 : s->L.route_edges);
    return TS_OK;
}
