// a6 + a7: batched placement objective and single-move deltas (section 5.2).
//
// The objective is linear in the slots of a candidate except for C_load, so every (layer)
// gets a small table indexed [expert][rank] that holds what one slot contributes:
//     w  = B[l,e] / r[l,e]                                   (rank load share,   PAPER.md:236)
//     c  = sum_s A[l,s,e] D[s,g] / r[l,e]                    (communication,     PAPER.md:244)
//     m  = M[l,e,g]                                          (migration,         PAPER.md:248)
// with the sign bit of c carrying "x0 already hosts e on g" (c >= 0 because A, D >= 0).
// C_mig = sum |x - x0| M = (M over the candidate's cells that x0 lacks) + (M over x0's cells -
// M over the cells both have) for binary x; exact for a scalar M, and with an M table the
// rounding is relative to sum of M over x0's cells.  r[l,e] is taken from x0: candidates place the
// same expert copies as x0 (R12); a candidate with another multiset of experts,
// an id out of range or an expert twice on one rank gets NaN.
//
// Scoring kernel: one block per (candidate chunk, layer); the layer's table sits in shared
// memory laid out [E][32] so that lane g only ever touches bank g (conflict-free gathers);
// lane <-> rank, so a rank's load is a lane-local sum and only the per-candidate reductions
// use shuffles.  Per-(candidate, layer) partials go to the workspace and a small finalize
// kernel reduces them over layers in fixed order.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

namespace gimbal {

constexpr int kMaxE = 256;
constexpr int kMaxG = 64;

struct PlaceTables {
    float2* wc;        // [L][E][GP]  {w, c with sign bit = member of x0}
    float* m;          // [L][E][GP]  M[l,e,g] (only when an M table is given)
    double* w_e;       // [L][E]      w in double (move deltas subtract nearly equal loads)
    uint32_t* hsum;    // [L]         multiset hash of x0's slot contents
    float* base_mig;   // [L]         sum over x0's cells of M
    double* sumB;      // [L]         sum_e B[l,e]
    int32_t* r;        // [L][E]      replica count in x0
    uint64_t* pmask;   // [L][E]      bit g set: x0 hosts e on rank g
    int32_t* bad;      // [1]         x0 invalid
};

__host__ __device__ inline int place_gp(int G) { return G < 32 ? 32 : G; }

__device__ __forceinline__ uint32_t slot_hash(uint32_t e) {
    uint32_t h = (e + 1u) * 0x9E3779B1u;
    h ^= h >> 15;
    return h * 0x85EBCA77u;
}

struct TableParams {
    int L, E, G, sp, S, counts_f32;
    const void* A; const void* B; const float* D; const float* M; float M_scalar;
    const int16_t* prev;
    PlaceTables t;
};

// one block per layer, 256 threads
__global__ void __launch_bounds__(256) place_tables_kernel(const TableParams p) {
    __shared__ int r_s[kMaxE];
    __shared__ unsigned long long pm_s[kMaxE];
    __shared__ float D_s[64 * 64];
    __shared__ int bad_s;
    __shared__ unsigned int hs_s;
    __shared__ float bm_s;
    __shared__ double sb_s;
    const int l = blockIdx.x, tid = threadIdx.x;
    const int NS = p.G * p.sp, GP = place_gp(p.G);
    const int16_t* pv = p.prev + (size_t)l * NS;
    if (tid == 0) { bad_s = 0; hs_s = 0; sb_s = 0.0; }
    for (int e = tid; e < p.E; e += 256) { r_s[e] = 0; pm_s[e] = 0ull; }
    for (int i = tid; i < p.S * p.G; i += 256) D_s[i] = p.D[i];
    __syncthreads();
    for (int j = tid; j < NS; j += 256) {
        const int e = pv[j], g = j / p.sp;
        if (e < 0 || e >= p.E) { bad_s = 1; continue; }
        atomicAdd(&r_s[e], 1);
        const unsigned long long old = atomicOr(&pm_s[e], 1ull << g);
        if ((old >> g) & 1ull) bad_s = 1;                         // twice on one rank
        atomicAdd(&hs_s, slot_hash((uint32_t)e));
    }
    if (tid == 0) {                                   // fixed order: bit-reproducible
        double bm = 0.0;
        for (int j = 0; j < NS; ++j) {
            const int e = pv[j], g = j / p.sp;
            if (e >= 0 && e < p.E) bm += p.M ? (double)p.M[((size_t)l * p.E + e) * p.G + g] : (double)p.M_scalar;
        }
        bm_s = (float)bm;
    }
    __syncthreads();
    for (int e = tid; e < p.E; e += 256) {
        if (r_s[e] < 1) bad_s = 1;
        const double b = p.counts_f32 ? (double)reinterpret_cast<const float*>(p.B)[(size_t)l * p.E + e]
                                      : (double)reinterpret_cast<const int32_t*>(p.B)[(size_t)l * p.E + e];
        atomicAdd(&sb_s, b);
        p.t.w_e[(size_t)l * p.E + e] = b / (double)max(r_s[e], 1);
        p.t.r[(size_t)l * p.E + e] = r_s[e];
        p.t.pmask[(size_t)l * p.E + e] = pm_s[e];
    }
    __syncthreads();
    // table entries; column gp of the table serves rank gp % G (replicated when G < 32)
    for (int i = tid; i < p.E * GP; i += 256) {
        const int e = i / GP, gp = i % GP, g = gp % p.G;
        float c = 0.0f;
        for (int s = 0; s < p.S; ++s) {
            const float a = p.counts_f32 ? reinterpret_cast<const float*>(p.A)[((size_t)l * p.S + s) * p.E + e]
                                         : (float)reinterpret_cast<const int32_t*>(p.A)[((size_t)l * p.S + s) * p.E + e];
            c = __fmaf_rn(a, D_s[s * p.G + g], c);
        }
        const float inv = 1.0f / (float)max(r_s[e], 1);
        c = fabsf(c * inv);
        const bool member = (pm_s[e] >> g) & 1ull;
        const float w = (float)p.t.w_e[(size_t)l * p.E + e];
        p.t.wc[((size_t)l * p.E + e) * GP + gp] = make_float2(w, member ? -c : c);   // -0.0f keeps the flag when c == 0
        if (p.M) p.t.m[((size_t)l * p.E + e) * GP + gp] = p.M[((size_t)l * p.E + e) * p.G + g];
    }
    if (tid == 0) {
        p.t.hsum[l] = hs_s;
        p.t.base_mig[l] = bm_s;
        p.t.sumB[l] = sb_s;
        if (bad_s) atomicOr(p.t.bad, 1);
    }
}

// ------------------------------------------------------------------------------------------
struct ScoreParams {
    int P, L, E, G, sp, chunk;          // chunk = candidates per block
    float M_scalar;
    int has_M;
    const int16_t* cand;                // [P,L,NS]
    PlaceTables t;
    float4* partial;                    // [P,L] {sum_g d_g^2, comm, mig, maxL}; NaN in .x if invalid
};

constexpr int kScoreThreads = 512;

template <int SP>
__device__ __forceinline__ void load_slots(const int16_t* g, int sp, int (&e)[16]) {
    // this lane's SP consecutive int16 slots
    if constexpr (SP == 8) {
        const uint4 q = __ldcs(reinterpret_cast<const uint4*>(g));
        e[0] = (int16_t)(q.x & 0xffff); e[1] = (int16_t)(q.x >> 16); e[2] = (int16_t)(q.y & 0xffff); e[3] = (int16_t)(q.y >> 16);
        e[4] = (int16_t)(q.z & 0xffff); e[5] = (int16_t)(q.z >> 16); e[6] = (int16_t)(q.w & 0xffff); e[7] = (int16_t)(q.w >> 16);
    } else if constexpr (SP == 4) {
        const uint2 q = __ldcs(reinterpret_cast<const uint2*>(g));
        e[0] = (int16_t)(q.x & 0xffff); e[1] = (int16_t)(q.x >> 16); e[2] = (int16_t)(q.y & 0xffff); e[3] = (int16_t)(q.y >> 16);
    } else {
#pragma unroll
        for (int j = 0; j < 16; ++j)
            if (j < sp) e[j] = __ldcs(g + j);
    }
}

// SP: compile-time slots per rank (0 = generic, runtime p.sp <= 16)
template <int SP>
__global__ void __launch_bounds__(kScoreThreads, 1) place_score_kernel(const ScoreParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int GP = place_gp(p.G);
    float2* wc_s = reinterpret_cast<float2*>(smem_raw);                       // [E][GP]
    float* m_s = reinterpret_cast<float*>(smem_raw + sizeof(float2) * (size_t)p.E * GP);   // [E][GP] (has_M)
    const int l = blockIdx.y;
    const int NS = p.G * p.sp;
    const int sp = SP > 0 ? SP : p.sp;
    {
        const uint4* src = reinterpret_cast<const uint4*>(p.t.wc + (size_t)l * p.E * GP);
        uint4* dst = reinterpret_cast<uint4*>(wc_s);
        for (int i = threadIdx.x; i < p.E * GP / 2; i += kScoreThreads) dst[i] = src[i];
        if (p.has_M) {
            const uint4* ms = reinterpret_cast<const uint4*>(p.t.m + (size_t)l * p.E * GP);
            uint4* md = reinterpret_cast<uint4*>(m_s);
            for (int i = threadIdx.x; i < p.E * GP / 4; i += kScoreThreads) md[i] = ms[i];
        }
    }
    __syncthreads();

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int upw = p.G < 32 ? 32 / p.G : 1;            // (candidate, layer) units per warp
    const int rpl = p.G > 32 ? p.G / 32 : 1;            // ranks per lane
    const int sub = p.G < 32 ? lane / p.G : 0;
    const int g0 = p.G < 32 ? lane % p.G : lane;
    const double Gd = (double)p.G;
    const double sumB = p.t.sumB[l];
    const uint32_t want_hash = p.t.hsum[l];
    const float base_mig = p.t.base_mig[l];
    const bool check_dup = NS > p.E;                    // with NS == E the multiset check already implies it

    const int p_begin = blockIdx.x * p.chunk, p_end = min(p.P, p_begin + p.chunk);
    for (int pc = p_begin + warp * upw; pc < p_end; pc += (kScoreThreads / 32) * upw) {
        const int cand = pc + sub;
        const bool active = cand < p_end;
        float sq = 0.0f, comm = 0.0f, mig_in = 0.0f, mig_kept = 0.0f, mx = -CUDART_INF_F;
        uint32_t hs = 0;
        int bad = 0;
        if (active) {
            const int16_t* row = p.cand + ((size_t)cand * p.L + l) * NS;
            for (int rr = 0; rr < rpl; ++rr) {
                const int g = g0 + rr * 32;
                int e[16];
                load_slots<SP>(row + g * sp, sp, e);
                float lg = 0.0f;
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    if (j < sp) {
                        int x = e[j];
                        if ((unsigned)x >= (unsigned)p.E) { bad = 1; x = 0; }
                        hs += slot_hash((uint32_t)x);
                        const int idx = x * GP + (p.G < 32 ? lane : g);
                        const float2 wc = wc_s[idx];
                        lg += wc.x;
                        comm += fabsf(wc.y);
                        const bool member = __float_as_int(wc.y) < 0;
                        const float mm = p.has_M ? m_s[idx] : p.M_scalar;
                        if (member) mig_kept += mm; else mig_in += mm;     // retained / entering cell of x0
                    }
                }
                if (check_dup) {
#pragma unroll
                    for (int a = 0; a < 16; ++a)
#pragma unroll
                        for (int b = a + 1; b < 16; ++b)
                            if (b < sp) bad |= (e[a] == e[b]);
                }
                const float d = (float)((double)lg * Gd - sumB);  // G*L_g - sum_g L_g, exact difference for integer counts
                sq = __fmaf_rn(d, d, sq);
                mx = fmaxf(mx, lg);
            }
        }
        // reduce over the lanes of this unit (segments of min(G,32) lanes)
        const int seg = p.G < 32 ? p.G : 32;
        for (int o = seg >> 1; o > 0; o >>= 1) {
            sq += __shfl_xor_sync(0xffffffffu, sq, o);
            comm += __shfl_xor_sync(0xffffffffu, comm, o);
            mig_in += __shfl_xor_sync(0xffffffffu, mig_in, o);
            mig_kept += __shfl_xor_sync(0xffffffffu, mig_kept, o);
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
            hs += __shfl_xor_sync(0xffffffffu, hs, o);
            bad |= __shfl_xor_sync(0xffffffffu, bad, o);
        }
        if (active && g0 == 0) {
            if (hs != want_hash) bad = 1;
            // C_mig = entering cells + (x0's cells - retained cells); exact for a scalar M
            float4 out = make_float4(sq, comm, mig_in + (base_mig - mig_kept), mx);
            if (bad) out.x = CUDART_NAN_F;
            p.partial[(size_t)cand * p.L + l] = out;
        }
    }
}

struct FinalizeParams {
    int P, L, G;
    float alpha, beta, gamma;
    const float4* partial;
    const int32_t* bad_prev;
    float* out;                         // [P,5]
    unsigned long long* best;           // workspace [1], init ~0ull
};

__device__ __forceinline__ uint32_t ordered_u32(float v) {
    const uint32_t b = __float_as_uint(v);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

__global__ void __launch_bounds__(256) place_finalize_kernel(const FinalizeParams p) {
    const int c = blockIdx.x * 256 + threadIdx.x;
    unsigned long long key = ~0ull;
    if (c < p.P) {
        double sq = 0.0, comm = 0.0, mig = 0.0, mx = 0.0;
        bool bad = *p.bad_prev != 0;
        for (int l = 0; l < p.L; ++l) {
            const float4 v = p.partial[(size_t)c * p.L + l];
            if (v.x != v.x) bad = true;
            sq += v.x; comm += v.y; mig += v.z; mx += v.w;
        }
        const double load = sq / ((double)p.G * (double)p.G);
        float* o = p.out + (size_t)c * 5;
        if (bad) {
            for (int i = 0; i < 5; ++i) o[i] = CUDART_NAN_F;
        } else {
            const float J = (float)((double)p.alpha * comm + (double)p.beta * load + (double)p.gamma * mig);
            o[0] = J; o[1] = (float)load; o[2] = (float)comm; o[3] = (float)mig; o[4] = (float)mx;
            key = ((unsigned long long)ordered_u32(J + 0.0f) << 32) | (unsigned)c;
        }
    }
    if (p.best) {
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long other = __shfl_xor_sync(0xffffffffu, key, o);
            key = other < key ? other : key;
        }
        if ((threadIdx.x & 31) == 0 && key != ~0ull) atomicMin(p.best, key);
    }
}

__global__ void best_to_index_kernel(const unsigned long long* best, int32_t* out, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = best[i] == ~0ull ? -1 : (int32_t)(best[i] & 0xffffffffull);
}

__global__ void fill_u64_kernel(unsigned long long* p, unsigned long long v, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

// ------------------------------------------------------------------------------------------
// a7 moves.  Per layer of `cur`: rank loads, the three largest of them, and which ranks host
// each expert; then one thread per move evaluates the closed-form deltas.
// ------------------------------------------------------------------------------------------
struct MovePrep {
    double* Lg;         // [L][G]
    double* top;        // [L][4]  three largest rank loads (value) ...
    int32_t* top_g;     // [L][4]  ... and their ranks
    uint64_t* cmask;    // [L][E]  bit g: cur hosts e on g
    int32_t* bad;       // [1]
};

struct MovePrepParams {
    int L, E, G, sp;
    const int16_t* cur;
    PlaceTables t;
    MovePrep mp;
};

__global__ void __launch_bounds__(256) move_prep_kernel(const MovePrepParams p) {
    __shared__ unsigned long long cm_s[kMaxE];
    __shared__ int cnt_s[kMaxE];
    __shared__ double lg_s[kMaxG];
    __shared__ int bad_s;
    const int l = blockIdx.x, tid = threadIdx.x, NS = p.G * p.sp;
    const int16_t* cu = p.cur + (size_t)l * NS;
    if (tid == 0) bad_s = 0;
    for (int e = tid; e < p.E; e += 256) { cm_s[e] = 0ull; cnt_s[e] = 0; }
    __syncthreads();
    for (int j = tid; j < NS; j += 256) {
        const int e = cu[j], g = j / p.sp;
        if (e < 0 || e >= p.E) { bad_s = 1; continue; }
        atomicAdd(&cnt_s[e], 1);
        if ((atomicOr(&cm_s[e], 1ull << g) >> g) & 1ull) bad_s = 1;
    }
    __syncthreads();
    for (int e = tid; e < p.E; e += 256) {
        if (cnt_s[e] != p.t.r[(size_t)l * p.E + e]) bad_s = 1;      // same expert copies as x0
        p.mp.cmask[(size_t)l * p.E + e] = cm_s[e];
    }
    if (tid < p.G) {
        double lg = 0.0;
        for (int j = 0; j < p.sp; ++j) {
            const int e = cu[tid * p.sp + j];
            if (e >= 0 && e < p.E) lg += p.t.w_e[(size_t)l * p.E + e];
        }
        lg_s[tid] = lg;
        p.mp.Lg[(size_t)l * p.G + tid] = lg;
    }
    __syncthreads();
    if (tid == 0) {
        double v[3] = {-CUDART_INF, -CUDART_INF, -CUDART_INF};
        int gi[3] = {-1, -1, -1};
        for (int g = 0; g < p.G; ++g) {
            const double x = lg_s[g];
            if (x > v[0]) { v[2] = v[1]; gi[2] = gi[1]; v[1] = v[0]; gi[1] = gi[0]; v[0] = x; gi[0] = g; }
            else if (x > v[1]) { v[2] = v[1]; gi[2] = gi[1]; v[1] = x; gi[1] = g; }
            else if (x > v[2]) { v[2] = x; gi[2] = g; }
        }
        for (int i = 0; i < 3; ++i) { p.mp.top[l * 4 + i] = v[i]; p.mp.top_g[l * 4 + i] = gi[i]; }
        if (bad_s) atomicOr(p.mp.bad, 1);
    }
}

struct MoveParams {
    int L, E, G, sp;
    long long n_moves;
    const int32_t* moves;               // [n,3] | nullptr (implicit all pairs)
    const int16_t* cur;
    float alpha, beta, gamma, M_scalar;
    int has_M;
    PlaceTables t;
    MovePrep mp;
    float* delta;                       // [n,5]
    unsigned long long* best;           // [L] | nullptr
};

__global__ void __launch_bounds__(256) move_delta_kernel(const MoveParams p) {
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= p.n_moves) return;
    const int NS = p.G * p.sp, GP = place_gp(p.G);
    int l, a, b;
    if (p.moves) {
        l = p.moves[i * 3]; a = p.moves[i * 3 + 1]; b = p.moves[i * 3 + 2];
    } else {
        const long long npairs = (long long)NS * (NS - 1) / 2;
        l = (int)(i / npairs);
        long long r = i % npairs;
        // canonical order: a outer, b inner, a < b.  Row a starts at a*NS - a*(a+1)/2.
        long long aa = (long long)floor(((2.0 * NS - 1.0) - sqrt((2.0 * NS - 1.0) * (2.0 * NS - 1.0) - 8.0 * (double)r)) * 0.5);
        if (aa < 0) aa = 0;
        while (aa * NS - aa * (aa + 1) / 2 > r) --aa;
        while ((aa + 1) * NS - (aa + 1) * (aa + 2) / 2 <= r) ++aa;
        a = (int)aa;
        b = (int)(r - (aa * NS - aa * (aa + 1) / 2)) + a + 1;
    }
    float* out = p.delta + i * 5;
    const bool bad_idx = l < 0 || l >= p.L || a < 0 || a >= NS || b < 0 || b >= NS;
    float dJ, dload, dcomm, dmig, dmax;
    bool nan = bad_idx || (*p.mp.bad != 0) || (*p.t.bad != 0);
    dJ = dload = dcomm = dmig = dmax = 0.0f;
    if (!nan) {
        const int16_t* cu = p.cur + (size_t)l * NS;
        const int e1 = cu[a], e2 = cu[b], g1 = a / p.sp, g2 = b / p.sp;
        if (g1 != g2 && e1 != e2) {
            const uint64_t cm1 = p.mp.cmask[(size_t)l * p.E + e1], cm2 = p.mp.cmask[(size_t)l * p.E + e2];
            if (((cm1 >> g2) & 1ull) || ((cm2 >> g1) & 1ull)) nan = true;      // second copy on a rank
            else {
                const float2* wc = p.t.wc + (size_t)l * p.E * GP;
                const float2 t11 = wc[e1 * GP + g1], t12 = wc[e1 * GP + g2], t21 = wc[e2 * GP + g1], t22 = wc[e2 * GP + g2];
                // loads in double: L1 - L2 and w2 - w1 subtract nearly equal numbers that can exceed 2^24
                const double w1 = p.t.w_e[(size_t)l * p.E + e1], w2 = p.t.w_e[(size_t)l * p.E + e2];
                const double L1 = p.mp.Lg[(size_t)l * p.G + g1], L2 = p.mp.Lg[(size_t)l * p.G + g2];
                const double dl = w2 - w1;                                    // moved onto g1
                dload = (float)(2.0 * dl * (L1 - L2) + 2.0 * dl * dl);        // the mean cancels
                dcomm = (fabsf(t12.y) - fabsf(t11.y)) + (fabsf(t21.y) - fabsf(t22.y));
                const float* mt = p.t.m + (size_t)l * p.E * GP;
                const float m11 = p.has_M ? mt[e1 * GP + g1] : p.M_scalar, m12 = p.has_M ? mt[e1 * GP + g2] : p.M_scalar;
                const float m21 = p.has_M ? mt[e2 * GP + g1] : p.M_scalar, m22 = p.has_M ? mt[e2 * GP + g2] : p.M_scalar;
                // leaving a cell x0 has: +M, leaving a cell x0 lacks: -M; entering: the opposite
                dmig = (__float_as_int(t11.y) < 0 ? m11 : -m11) + (__float_as_int(t12.y) < 0 ? -m12 : m12) +
                       (__float_as_int(t22.y) < 0 ? m22 : -m22) + (__float_as_int(t21.y) < 0 ? -m21 : m21);
                const double n1 = L1 + dl, n2 = L2 - dl;
                double rest = -CUDART_INF;
                for (int q = 0; q < 3; ++q) {
                    const int tg = p.mp.top_g[l * 4 + q];
                    if (tg >= 0 && tg != g1 && tg != g2) { rest = p.mp.top[l * 4 + q]; break; }
                }
                dmax = (float)(fmax(fmax(n1, n2), rest) - p.mp.top[l * 4]);
                dJ = p.alpha * dcomm + p.beta * dload + p.gamma * dmig;
            }
        }
    }
    if (nan) dJ = dload = dcomm = dmig = dmax = CUDART_NAN_F;
    out[0] = dJ; out[1] = dload; out[2] = dcomm; out[3] = dmig; out[4] = dmax;
    if (p.best && !nan) {
        const unsigned long long key = ((unsigned long long)ordered_u32(dJ + 0.0f) << 32) | (unsigned long long)(uint32_t)(i & 0xffffffffll);
        atomicMin(p.best + l, key);
    }
}

}  // namespace gimbal
