// NEXT-2: Algorithm 1, Global DP Engine Scheduling (section 4.3; readings DESIGN.md R19),
// batched over B independent scheduler instances: one warp per instance, lane <-> engine (two engines per
// lane when N > 32), the R requests of an instance in order.  Decisions in IEEE double, one rounding per
// operation, so the chosen engines are a pure function of the inputs (bit-exact against the oracle).
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

namespace gimbal {

struct SchedParams {
    int B, N, R;
    double high_kv, large_gap, lambda_kv, lambda_moe, close_frac;
    const float* trace;        // [B,N,4] {kv, pre_rem, wait, moe}
    const uint8_t* complete;   // [B] | nullptr (all complete)
    const float* req_len;      // [B,R]
    double* comp;              // [B,N] inout
    int32_t* rr;               // [B] inout
    int32_t* engine;           // [B,R] out
};

struct SchedKey { double a, b; int i; };     // lexicographic (a, b, i)
__device__ __forceinline__ bool sched_before(const SchedKey& x, const SchedKey& y) {
    return x.a < y.a || (x.a == y.a && (x.b < y.b || (x.b == y.b && x.i < y.i)));
}
__device__ __forceinline__ SchedKey sched_warp_min(SchedKey k) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        SchedKey t;
        t.a = __shfl_xor_sync(0xffffffffu, k.a, o);
        t.b = __shfl_xor_sync(0xffffffffu, k.b, o);
        t.i = __shfl_xor_sync(0xffffffffu, k.i, o);
        if (sched_before(t, k)) k = t;
    }
    return k;
}

constexpr int kSchedWarps = 4;

__global__ void __launch_bounds__(kSchedWarps * 32) select_engines_kernel(const SchedParams p) {
    const int b = blockIdx.x * kSchedWarps + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (b >= p.B) return;
    const float* tr = p.trace + (size_t)b * p.N * 4;
    double kv[2], base[2], comp[2];
    bool have[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const int i = lane + 32 * q;
        have[q] = i < p.N;
        kv[q] = base[q] = comp[q] = 0.0;
        if (have[q]) {
            const float4 t = *reinterpret_cast<const float4*>(tr + i * 4);
            kv[q] = (double)t.x;
            base[q] = __dadd_rn((double)t.y, (double)t.z);             // pre_rem + wait
            comp[q] = p.comp[(size_t)b * p.N + i];
        }
    }
    const bool complete = p.complete ? p.complete[b] != 0 : true;
    int rr = p.rr[b];
    rr = ((rr % p.N) + p.N) % p.N;                                       // the pointer counts modulo N (R19)
    // KV rule (lines 6-9): argmin / argmax of kv, lowest index on ties; the same for every request of the call
    SchedKey kmin{CUDART_INF, 0.0, INT32_MAX}, kmax{CUDART_INF, 0.0, INT32_MAX};
#pragma unroll
    for (int q = 0; q < 2; ++q)
        if (have[q]) {
            const SchedKey a{kv[q], 0.0, lane + 32 * q}, c{-kv[q], 0.0, lane + 32 * q};
            if (sched_before(a, kmin)) kmin = a;
            if (sched_before(c, kmax)) kmax = c;
        }
    kmin = sched_warp_min(kmin);
    kmax = sched_warp_min(kmax);
    const double kvmin = kmin.a, kvmax = -kmax.a;
    const bool kv_rule = kvmax > p.high_kv && __dsub_rn(kvmax, kvmin) > p.large_gap;
    double pk[2], pm[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const int i = lane + 32 * q;
        pk[q] = __dmul_rn(p.lambda_kv, kv[q]);
        pm[q] = have[q] ? __dmul_rn(p.lambda_moe, (double)tr[i * 4 + 3]) : 0.0;
    }
    for (int r = 0; r < p.R; ++r) {
        const double len = (double)p.req_len[(size_t)b * p.R + r];
        int pick;
        if (!complete) {
            pick = rr; rr = (rr + 1) % p.N;
        } else if (kv_rule) {
            pick = kmin.i;
        } else {
            SchedKey best{CUDART_INF, 0.0, INT32_MAX}, lo{CUDART_INF, 0.0, 0}, hi{CUDART_INF, 0.0, 0};
#pragma unroll
            for (int q = 0; q < 2; ++q)
                if (have[q]) {
                    const double sc = __dadd_rn(__dadd_rn(__dadd_rn(base[q], comp[q]), pk[q]), pm[q]);
                    const SchedKey k{sc, kv[q], lane + 32 * q};
                    if (sched_before(k, best)) best = k;
                    if (sc < lo.a) lo.a = sc;
                    if (-sc < hi.a) hi.a = -sc;
                }
            best = sched_warp_min(best);
            lo = sched_warp_min(lo);
            hi = sched_warp_min(hi);
            const double delta = __dsub_rn(-hi.a, lo.a);
            if (delta < __dmul_rn(p.close_frac, len)) { pick = rr; rr = (rr + 1) % p.N; }
            else pick = best.i;
        }
#pragma unroll
        for (int q = 0; q < 2; ++q)
            if (lane + 32 * q == pick) comp[q] = __dadd_rn(comp[q], len);
        if (lane == 0) p.engine[(size_t)b * p.R + r] = pick;
    }
#pragma unroll
    for (int q = 0; q < 2; ++q)
        if (have[q]) p.comp[(size_t)b * p.N + lane + 32 * q] = comp[q];
    if (lane == 0) p.rr[b] = rr;
}

// ------------------------------------------------------------------------------------------
// Algorithm 2, SJF with aging (R20), batched over B waiting queues: one block per queue,
// position of request j = number of requests that come before it in the total order (aged first and oldest
// first, then shortest prefill, then oldest, then input position) -- a counting rank, deterministic, no sort.
// The waiting time uses the same fp32 subtraction as the oracle.
// ------------------------------------------------------------------------------------------
struct QueueParams {
    int B, Q;                      // queues, capacity of a queue (row pitch)
    float now, theta_age;
    const float* arrival;          // [B,Q]
    const int32_t* prefill;        // [B,Q]
    const int32_t* qlen;           // [B]
    int32_t* order;                // [B,Q]; entries past qlen are -1
};

constexpr int kQueueThreads = 256;
constexpr int kQueueMax = 2048;

__global__ void __launch_bounds__(kQueueThreads) order_queues_kernel(const QueueParams p) {
    __shared__ float arr_s[kQueueMax];
    __shared__ int32_t pre_s[kQueueMax];
    const int b = blockIdx.x;
    const int n = min(max(p.qlen[b], 0), p.Q);
    for (int j = threadIdx.x; j < n; j += kQueueThreads) {
        const float a = p.arrival[(size_t)b * p.Q + j];
        arr_s[j] = a != a ? CUDART_INF_F : a;                               // a NaN arrival is the youngest request (R20)
        pre_s[j] = p.prefill[(size_t)b * p.Q + j];
    }
    for (int j = n + threadIdx.x; j < p.Q; j += kQueueThreads) p.order[(size_t)b * p.Q + j] = -1;
    __syncthreads();
    for (int j = threadIdx.x; j < n; j += kQueueThreads) {
        const float aj = arr_s[j];
        const int pj = pre_s[j];
        const bool aged_j = __fsub_rn(p.now, aj) >= p.theta_age;
        int pos = 0;
        for (int i = 0; i < n; ++i) {
            const float ai = arr_s[i];
            const int pi = pre_s[i];
            const bool aged_i = __fsub_rn(p.now, ai) >= p.theta_age;
            bool before;
            if (aged_i != aged_j) before = aged_i;
            else if (!aged_i && pi != pj) before = pi < pj;
            else if (ai != aj) before = ai < aj;
            else before = i < j;
            pos += before;
        }
        p.order[(size_t)b * p.Q + pos] = j;
    }
}

}  // namespace gimbal
