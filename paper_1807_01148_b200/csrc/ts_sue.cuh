// ts_sue.cuh -- static user equilibrium by Frank-Wolfe with BPR times (
// PAPER.md:307-338 section 5.3, Eq. 6; Eq. 3 with alpha = 0.15, beta = 4).
//
// The paper's comparator workload.  Per iteration: BPR times -> integer routing weights (R43) ->
// one shortest-path tree per origin (k_rr_sssp of ts_reroute.cuh) -> all-or-nothing loading with
// integer atomics (R44: trips are integers, so y is exact and order-independent) -> step length by
// bisection on the directional derivative (fp64 block sums, added up in a fixed order on the host)
// -> x += a (y - x).  fp64 throughout, one rounding per written operation (-fmad=false).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ts {

constexpr uint32_t kSueBlocks = 148, kSueThreads = 256;

// Eq. 3 with beta = 4 (reading R42: two squarings)
__device__ __forceinline__ double bpr_time(double t0, double cap, double x, double alpha) {
    const double r = x / cap;
    const double r2 = r * r;
    return t0 * (1.0 + alpha * (r2 * r2));
}

// t[e] = BPR time at flow x[e] (x == nullptr: free flow) and the integer weight the trees are grown on
__global__ void k_sue_times(uint32_t E, const double* t0, const double* cap, const double* x, double alpha,
                            double scale, double* t, uint32_t* w) {
    for (uint32_t e = blockIdx.x * blockDim.x + threadIdx.x; e < E; e += gridDim.x * blockDim.x) {
        const double te = x ? bpr_time(t0[e], cap[e], x[e], alpha) : t0[e];
        t[e] = te;
        double q = rint(te * scale);                    // round half to even, like numpy.rint
        q = q < 1.0 ? 1.0 : (q > 1048576.0 ? 1048576.0 : q);
        w[e] = (uint32_t)q;
    }
}

// all-or-nothing: every OD pair's trips on its shortest path, walked back from the destination
__global__ void k_sue_aon(uint32_t n_od, const uint32_t* od_origin, const uint32_t* od_dest, const uint32_t* od_trips,
                          const uint32_t* od_src, const uint32_t* pred, uint32_t N, const uint32_t* edge_from,
                          unsigned long long* y) {
    for (uint32_t q = blockIdx.x * blockDim.x + threadIdx.x; q < n_od; q += gridDim.x * blockDim.x) {
        const uint32_t o = od_origin[q];
        uint32_t v = od_dest[q];
        const uint32_t* row = pred + (size_t)od_src[q] * N;
        if (o == v || row[v] == 0xFFFFFFFFu) continue;
        const unsigned long long trips = od_trips[q];
        for (uint32_t n = 0; v != o && n <= N; n++) { const uint32_t e = row[v]; atomicAdd(y + e, trips); v = edge_from[e]; }
    }
}

__device__ __forceinline__ double block_sum_f64(double v, double* sh) {
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0) for (uint32_t w = 0; w < blockDim.x / 32; w++) s += sh[w];
    __syncthreads();
    return s;
}

// mode 0: g(a) = sum (y - x) t(x + a (y - x))      -> out[block]
// mode 1: f(x) = sum t0 (x + alpha x^5 / (5 c^4))  -> out[block]
// mode 2: sum x t(x) -> out[block], sum y t(x) -> out[gridDim.x + block]
__global__ void __launch_bounds__(kSueThreads) k_sue_reduce(int mode, uint32_t E, const double* t0, const double* cap,
                                                          const double* x, const unsigned long long* y, double a,
                                                          double alpha, double* out) {
    __shared__ double sh[kSueThreads / 32];
    double s0 = 0.0, s1 = 0.0;
    for (uint32_t e = blockIdx.x * blockDim.x + threadIdx.x; e < E; e += gridDim.x * blockDim.x) {
        const double xe = x[e];
        if (mode == 0) {
            const double d = (double)y[e] - xe;
            s0 += d * bpr_time(t0[e], cap[e], xe + a * d, alpha);
        } else if (mode == 1) {
            const double r = xe / cap[e];
            const double r2 = r * r;
            s0 += t0[e] * (xe + (alpha / 5.0) * (xe * (r2 * r2)));
        } else {
            const double te = bpr_time(t0[e], cap[e], xe, alpha);
            s0 += xe * te;
            s1 += (double)y[e] * te;
        }
    }
    s0 = block_sum_f64(s0, sh);
    if (mode == 2) s1 = block_sum_f64(s1, sh);
    if (threadIdx.x == 0) { out[blockIdx.x] = s0; if (mode == 2) out[gridDim.x + blockIdx.x] = s1; }
}

// x = y (first = 1) or x += a (y - x)
__global__ void k_sue_update(uint32_t E, double* x, const unsigned long long* y, double a, int first) {
    for (uint32_t e = blockIdx.x * blockDim.x + threadIdx.x; e < E; e += gridDim.x * blockDim.x) {
        const double ye = (double)y[e];
        x[e] = first ? ye : x[e] + a * (ye - x[e]);
    }
}

}  // namespace ts
