// NEXT-1: the online greedy placement heuristic of PAPER.md:260-268 (section 5.3) on device.
// One block per layer (layers are independent):
//   1. replica counts / rank masks of x0, per-expert volume and load share, the table
//      c[e][g] = sum_s A[l,s,e] D[s,g] / r (double, s ascending, one rounding per operation)
//   2. hotness ranking of the NS items (slot contents of x0) by counting: position of item j =
//      #{items before j in (hot desc, expert asc, slot asc)}
//   3. warp 0 walks the items in that order; lane <-> rank (two ranks per lane when G = 64)
//      scores its rank  S = ((alpha*c) + (beta*(Lcur+b))) + (gamma*m)  in IEEE double, and a
//      butterfly takes the lexicographic minimum of (S, migrates, fill, rank) -- the paper's
//      tie-break "avoid migration, then less-filled ranks", then rank index.
// The decision arithmetic is double on both sides (R17), spelled with __dmul_rn /
// __dadd_rn / __ddiv_rn so that nothing is contracted into an FMA.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

namespace gimbal {

struct GreedyParams {
    int L, E, G, sp, S, counts_f32;
    const void* A; const void* B; const float* D; const float* M; float M_scalar;
    float alpha, beta, gamma;
    const int16_t* prev;            // x0 [L,NS]
    int16_t* out;                   // [L,NS]
    int32_t* status;                // [1] | nullptr: bit 1 set when a layer failed
};

constexpr int kGreedyThreads = 256;

__host__ __device__ inline size_t greedy_smem_bytes(int E, int G, int NS) {
    return sizeof(double) * ((size_t)E * G + 2 * (size_t)E + NS + G) + sizeof(unsigned long long) * 2 * (size_t)E +
           sizeof(int) * ((size_t)E + NS + 8) + sizeof(int16_t) * ((size_t)NS + 8);
}

struct GreedyKey {
    double s;       // score
    int t;          // (migrates << 24) | (fill << 8) | rank ; INT_MAX when infeasible
};
__device__ __forceinline__ bool greedy_before(const GreedyKey& a, const GreedyKey& b) {
    return a.s < b.s || (a.s == b.s && a.t < b.t);
}

__global__ void __launch_bounds__(kGreedyThreads) greedy_place_kernel(const GreedyParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int NS = p.G * p.sp, l = blockIdx.x, tid = threadIdx.x;
    double* cD = reinterpret_cast<double*>(smem_raw);                 // [E][G]
    double* bD = cD + (size_t)p.E * p.G;                              // [E]  B / r
    double* vol = bD + p.E;                                           // [E]  sum_s A
    double* hot = vol + p.E;                                          // [NS]
    double* Lcur = hot + NS;                                          // [G]
    unsigned long long* pm_s = reinterpret_cast<unsigned long long*>(Lcur + p.G);   // [E] x0 hosts e on g
    unsigned long long* has_s = pm_s + p.E;                           // [E] this pass placed e on g
    int* r_s = reinterpret_cast<int*>(has_s + p.E);                   // [E]
    int* order = r_s + p.E;                                           // [NS]
    int* flag = order + NS;                                           // [8]
    int16_t* pv = reinterpret_cast<int16_t*>(flag + 8);               // [NS]

    const int16_t* prev = p.prev + (size_t)l * NS;
    int16_t* out = p.out + (size_t)l * NS;
    if (tid == 0) flag[0] = 0;
    for (int e = tid; e < p.E; e += kGreedyThreads) { r_s[e] = 0; pm_s[e] = 0ull; has_s[e] = 0ull; }
    __syncthreads();
    for (int j = tid; j < NS; j += kGreedyThreads) {
        const int e = prev[j], g = j / p.sp;
        pv[j] = (int16_t)e;
        if (e < 0 || e >= p.E) { flag[0] = 1; continue; }
        atomicAdd(&r_s[e], 1);
        if ((atomicOr(&pm_s[e], 1ull << g) >> g) & 1ull) flag[0] = 1;          // twice on one rank
    }
    __syncthreads();
    for (int e = tid; e < p.E; e += kGreedyThreads) {
        if (r_s[e] < 1) flag[0] = 1;
        const double r = (double)max(r_s[e], 1);
        double v = 0.0;
        for (int s = 0; s < p.S; ++s) {
            const size_t i = ((size_t)l * p.S + s) * p.E + e;
            v = __dadd_rn(v, p.counts_f32 ? (double)reinterpret_cast<const float*>(p.A)[i] : (double)reinterpret_cast<const int32_t*>(p.A)[i]);
        }
        const double b = p.counts_f32 ? (double)reinterpret_cast<const float*>(p.B)[(size_t)l * p.E + e]
                                      : (double)reinterpret_cast<const int32_t*>(p.B)[(size_t)l * p.E + e];
        bD[e] = __ddiv_rn(b, r);
        vol[e] = __ddiv_rn(__dadd_rn(b, v), r);                                   // hotness of one copy
    }
    for (int i = tid; i < p.E * p.G; i += kGreedyThreads) {
        const int e = i / p.G, g = i - e * p.G;
        double c = 0.0;
        for (int s = 0; s < p.S; ++s) {
            const size_t ia = ((size_t)l * p.S + s) * p.E + e;
            const double a = p.counts_f32 ? (double)reinterpret_cast<const float*>(p.A)[ia] : (double)reinterpret_cast<const int32_t*>(p.A)[ia];
            c = __dadd_rn(c, __dmul_rn(a, (double)p.D[s * p.G + g]));
        }
        cD[i] = __ddiv_rn(c, (double)max(r_s[e], 1));
    }
    __syncthreads();
    const bool bad = flag[0] != 0;
    if (!bad) {
        for (int j = tid; j < NS; j += kGreedyThreads) hot[j] = vol[pv[j]];
    }
    __syncthreads();
    if (!bad) {
        // ranking by counting under the total order (hot desc, expert asc, slot asc)
        for (int j = tid; j < NS; j += kGreedyThreads) {
            const double hj = hot[j];
            const int ej = pv[j];
            int pos = 0;
            for (int i = 0; i < NS; ++i) {
                const double hi = hot[i];
                const int ei = pv[i];
                pos += (hi > hj) || (hi == hj && (ei < ej || (ei == ej && i < j)));
            }
            order[pos] = j;
        }
    }
    __syncthreads();
    if (tid >= 32) return;

    // ---- greedy assignment by warp 0 ----
    const int lane = tid;
    const int rpl = p.G > 32 ? 2 : 1;
    const double alpha = (double)p.alpha, beta = (double)p.beta, gamma = (double)p.gamma;
    double Lc[2] = {0.0, 0.0};
    int fill[2] = {0, 0};
    bool stuck = bad;
    for (int i = 0; i < NS && !stuck; ++i) {
        const int e = pv[order[i]];
        const double b = bD[e];
        const unsigned long long has = has_s[e], pm = pm_s[e];
        GreedyKey best{CUDART_INF, INT32_MAX};
#pragma unroll
        for (int rr = 0; rr < 2; ++rr) {
            const int g = lane + rr * 32;
            if (rr < rpl && g < p.G && fill[rr] < p.sp && !((has >> g) & 1ull)) {
                const int mig = ((pm >> g) & 1ull) ? 0 : 1;
                const double m = mig ? (p.M ? (double)p.M[((size_t)l * p.E + e) * p.G + g] : (double)p.M_scalar) : 0.0;
                const double load = __dadd_rn(Lc[rr], b);
                const double sc = __dadd_rn(__dadd_rn(__dmul_rn(alpha, cD[e * p.G + g]), __dmul_rn(beta, load)), __dmul_rn(gamma, m));
                const GreedyKey k{sc, (mig << 24) | (fill[rr] << 8) | g};
                if (greedy_before(k, best)) best = k;
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            GreedyKey other;
            other.s = __shfl_xor_sync(0xffffffffu, best.s, o);
            other.t = __shfl_xor_sync(0xffffffffu, best.t, o);
            if (greedy_before(other, best)) best = other;
        }
        if (best.t == INT32_MAX) { stuck = true; break; }
        const int bg = best.t & 0xff;
#pragma unroll
        for (int rr = 0; rr < 2; ++rr) {
            if (lane + rr * 32 == bg) {
                out[bg * p.sp + fill[rr]] = (int16_t)e;
                fill[rr] += 1;
                Lc[rr] = __dadd_rn(Lc[rr], b);
            }
        }
        if (lane == 0) has_s[e] = has | (1ull << bg);
        __syncwarp();
    }
    if (stuck) {
        for (int j = lane; j < NS; j += 32) out[j] = -1;
        if (lane == 0 && p.status) atomicOr(p.status, 2);
    }
}

}  // namespace gimbal
