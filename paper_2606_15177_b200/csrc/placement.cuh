// a6 + a7: batched placement objective and single-move deltas (section 5.2).
//
// The objective is linear in the slots of a candidate except for C_load, so every layer gets a
// small table indexed [expert][rank] that holds what one slot contributes:
//     w  = B[l,e] / r[l,e]                                   (rank load share,   PAPER.md:236)
//     c  = sum_s A[l,s,e] D[s,g] / r[l,e]                    (communication,     PAPER.md:244)
//     m  = M[l,e,g]                                          (migration,         PAPER.md:248)
// with the sign bit of c carrying "x0 already hosts e on g" (c >= 0 because A, D >= 0).
//
// Three kernels share the work (K4):
//   place_score_kernel   the throughput kernel.  It assumes what place_check_kernel proves: the
//                        candidate is valid and hosts as many copies of every expert as x0 (so the
//                        tables' r = r0 is the candidate's r).  One block per (candidate chunk,
//                        layer); the layer's table sits in shared memory laid out [E][32] so that
//                        lane g only ever touches bank g (conflict-free gathers); lane <-> rank, so
//                        a rank's load is a lane-local sum and only the per-candidate reductions
//                        use shuffles.  Five instructions per slot with a scalar M.
//   place_check_kernel   exact validation (R12): a warp builds the candidate's binary
//                        x[e,g] as per-expert rank masks in shared memory (one atomicOr per slot:
//                        the returned word tells "twice on one rank", its popcount is r[l,e]).
//                        Invalid -> NaN; valid with other replica counts than x0 -> scored right here
//                        with the candidate's own r (the plain definition, from global memory);
//                        valid with x0's counts -> left to place_score_kernel.
//   place_finalize_kernel reduces the per-(candidate, layer) partials over layers in fixed order.
// C_mig = sum M |x - x0| is accumulated directly from the cells that enter (candidate slot on a cell
// x0 lacks) and the cells that leave (x0 slot whose cell the candidate lacks): no subtraction of
// nearly equal sums, so a candidate equal to x0 gives exactly 0.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "ptx.cuh"

namespace gimbal {

constexpr int kMaxE = 256;
constexpr int kMaxG = 64;

struct PlaceTables {
    float2* wc;        // [L][GP/32][E][32]  {w, c with sign bit = member of x0}
    float* c_s;        // [L][GP/32][E][32]  the c half of wc alone, and
    float* w_f;        // [L][E]             its w half: what place_score_tma_kernel stages (half the bytes)
    float* m;          // [L][GP/32][E][32]  M[l,e,g]                                   (M table only)
    uint32_t* mu;      // [L][GP/32][E][32]  scoring word: float bits of M where x0 lacks the cell, else
                       //                    0x80000000 | 1 << (position of e among x0's slots of rank g)   (M table only)
    float* mx0;        // [L][NS]     M of x0's own cell of every slot                  (M table only)
    float* c_raw;      // [L][E][G]   sum_s A D, not divided by r   (place_check_kernel's own scoring)
    double* b_raw;     // [L][E]      B as double                   (same)
    double* w_e;       // [L][E]      w in double (move deltas subtract nearly equal loads)
    double* sumB;      // [L]         sum_e B[l,e]
    int32_t* r;        // [L][E]      replica count in x0
    uint64_t* pmask;   // [L][E]      bit g set: x0 hosts e on rank g
    int32_t* bad;      // [1]         x0 invalid
};

__host__ __device__ inline int place_gp(int G) { return G < 32 ? 32 : G; }
// cell (expert e, table column gp) of a layer's [GP/32][E][32] table; column gp serves rank gp % G
__host__ __device__ inline size_t tab_idx(int E, int e, int gp) { return ((size_t)(gp >> 5) * E + e) * 32 + (gp & 31); }

struct TableParams {
    int L, E, G, sp, S, counts_f32;
    const void* A; const void* B; const float* D; const float* M; float M_scalar;
    const int16_t* prev;
    PlaceTables t;
};

// fixed-order block sum of one double per thread (256 threads): bit-reproducible
__device__ __forceinline__ double block_sum_256(double v, double* red) {
    red[threadIdx.x] = v;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    const double r = red[0];
    __syncthreads();
    return r;
}

constexpr int kTableSplit = 4;      // blocks per layer (the [E][G'] cells are split between them)

// grid (L, kTableSplit), 256 threads.  Every block rebuilds the layer's replica counts / rank
// masks of x0 (cheap); block y = 0 also writes the per-layer scalars and the per-slot entries.
__global__ void __launch_bounds__(256) place_tables_kernel(const TableParams p) {
    __shared__ int r_s[kMaxE];
    __shared__ unsigned long long pm_s[kMaxE];
    __shared__ float D_s[64 * 64];
    __shared__ double red_s[256];
    __shared__ int bad_s;
    extern __shared__ __align__(16) unsigned char tab_smem[];
    float* A_s = reinterpret_cast<float*>(tab_smem);              // [S][E] this layer's counts as fp32
    const int l = blockIdx.x, tid = threadIdx.x;
    const int NS = p.G * p.sp, GP = place_gp(p.G);
    const int16_t* pv = p.prev + (size_t)l * NS;
    if (tid == 0) bad_s = 0;
    for (int e = tid; e < p.E; e += 256) { r_s[e] = 0; pm_s[e] = 0ull; }
    for (int i = tid; i < p.S * p.G; i += 256) D_s[i] = p.D[i];
    for (int i = tid; i < p.S * p.E; i += 256)
        A_s[i] = p.counts_f32 ? reinterpret_cast<const float*>(p.A)[(size_t)l * p.S * p.E + i]
                              : (float)reinterpret_cast<const int32_t*>(p.A)[(size_t)l * p.S * p.E + i];
    __syncthreads();
    for (int j = tid; j < NS; j += 256) {
        const int e = pv[j], g = j / p.sp;
        if (e < 0 || e >= p.E) { bad_s = 1; continue; }
        atomicAdd(&r_s[e], 1);
        const unsigned long long old = atomicOr(&pm_s[e], 1ull << g);
        if ((old >> g) & 1ull) bad_s = 1;                         // twice on one rank
    }
    __syncthreads();
    const size_t tab = (size_t)l * (GP / 32) * p.E * 32;
    if (blockIdx.y == 0) {
        double sb = 0.0;
        for (int e = tid; e < p.E; e += 256) {
            if (r_s[e] < 1) bad_s = 1;
            const double b = p.counts_f32 ? (double)reinterpret_cast<const float*>(p.B)[(size_t)l * p.E + e]
                                          : (double)reinterpret_cast<const int32_t*>(p.B)[(size_t)l * p.E + e];
            sb += b;
            p.t.b_raw[(size_t)l * p.E + e] = b;
            p.t.w_e[(size_t)l * p.E + e] = b / (double)max(r_s[e], 1);
            p.t.w_f[(size_t)l * p.E + e] = (float)(b / (double)max(r_s[e], 1));
            p.t.r[(size_t)l * p.E + e] = r_s[e];
            p.t.pmask[(size_t)l * p.E + e] = pm_s[e];
        }
        const double sb_tot = block_sum_256(sb, red_s);
        if (tid == 0) {
            p.t.sumB[l] = sb_tot;
            if (bad_s) atomicOr(p.t.bad, 1);
        }
        if (p.M) {
            // x0's own cells: the scoring word names the slot's position inside its rank, mx0 holds its M
            for (int j = tid; j < NS; j += 256) {
                const int e = pv[j], g = j / p.sp;
                if (e < 0 || e >= p.E) { p.t.mx0[(size_t)l * NS + j] = 0.0f; continue; }
                p.t.mx0[(size_t)l * NS + j] = p.M[((size_t)l * p.E + e) * p.G + g];
                for (int gp = g; gp < GP; gp += p.G) p.t.mu[tab + tab_idx(p.E, e, gp)] = 0x80000000u | (1u << (j - g * p.sp));
            }
        }
    }
    // table entries; column gp of the table serves rank gp % G (replicated when G < 32)
    const int cells = p.E * GP, per = (cells + kTableSplit - 1) / kTableSplit;
    const int i_end = min(cells, (int)(blockIdx.y + 1) * per);
    for (int i = blockIdx.y * per + tid; i < i_end; i += 256) {
        const int e = i / GP, gp = i % GP, g = gp % p.G;
        float c = 0.0f;
        for (int s = 0; s < p.S; ++s) c = __fmaf_rn(A_s[s * p.E + e], D_s[s * p.G + g], c);
        if (gp < p.G) p.t.c_raw[((size_t)l * p.E + e) * p.G + g] = fabsf(c);
        const int re = max(r_s[e], 1);
        const float inv = 1.0f / (float)re;
        c = fabsf(c * inv);
        const bool member = (pm_s[e] >> g) & 1ull;
        const double b = p.counts_f32 ? (double)reinterpret_cast<const float*>(p.B)[(size_t)l * p.E + e]
                                      : (double)reinterpret_cast<const int32_t*>(p.B)[(size_t)l * p.E + e];
        const float w = (float)(b / (double)re);
        const size_t at = tab + tab_idx(p.E, e, gp);
        p.t.wc[at] = make_float2(w, member ? -c : c);   // -0.0f keeps the flag when c == 0
        p.t.c_s[at] = member ? -c : c;
        if (p.M) {
            const float mm = p.M[((size_t)l * p.E + e) * p.G + g];
            p.t.m[at] = mm;
            if (!member) p.t.mu[at] = __float_as_uint(fabsf(mm));
        }
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
    uint8_t* status;                    // [L,P] verdicts of the fused validation (kCheck): 0 same copies as x0, 1 invalid, 2 other replica counts
    int force_general;                  // tests: verdict 2 for every valid candidate
    uint32_t zero;                      // 0 at run time, opaque to the compiler: place_score_tma_kernel's ordering dependency
};

constexpr int kScoreThreads = 512;

// reduce (sq, comm) over the SEG lanes of a unit with a transposed butterfly (the first step folds
// both values into one register); returns comm's total, leaves sq's total in `sq` on the unit's lanes
// with bit SEG/2 clear
template <int SEG>
__device__ __forceinline__ float reduce_pair(float& sq, float comm, int lane, int sub) {
    if constexpr (SEG > 1) {
        constexpr int h = SEG >> 1;
        const bool up = (lane & h) != 0;
        float v = (up ? comm : sq) + __shfl_xor_sync(0xffffffffu, up ? sq : comm, h);
#pragma unroll
        for (int o = h >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        const float commt = __shfl_sync(0xffffffffu, v, sub * SEG + h);
        sq = v;
        return commt;
    } else {
        return comm;
    }
}

// Throughput kernel for the five configuration shapes: compile-time (slots per rank, ranks, experts).  Slot ids
// arrive as aligned 32-bit words (two per word; ranks with an odd slot count are realigned with a
// funnel shift); one PRMT turns an id into the byte offset of its table cell (id << 8 | lane * 8),
// one 8-byte shared load fetches {w, c}, two adds and one shift-add (x0 membership) finish the slot.
// Ids are masked to the table, so a row that place_check_kernel would reject cannot fault here.
// A warp pass takes two candidates per unit: their instruction streams interleave and one transposed
// butterfly reduces both; the rows of the next pass are prefetched into the other half of a register
// ping-pong.  G*L_g - sum_e B is one fp32 FMA against the high part of sum_e B plus one subtraction of
// the low part: exact whenever the difference is representable (integer counts), R11.
constexpr int kScoreU = 2;

// kCheck (the default call on these shapes): the exact validation of place_check_kernel runs on the ids while they are in registers --
// one atomicOr per slot into the unit's x[e, .] rank masks in shared memory, read back (and cleared) by 16-byte loads, popcounts compared
// with x0's replica counts -- and the verdict decides what is stored: NaN (invalid), the scores (same copies as x0), or the scores plus
// verdict 2 for place_own_r_kernel to replace (valid, other replica counts).
inline size_t place_score_mask_bytes(int G, int E) {
    const int upw = G < 32 ? 32 / G : 1, h = G > 32 ? G / 32 : 1;
    return sizeof(uint32_t) * (size_t)(kScoreThreads / 32) * upw * 2 * h * E;       // [warps][units per warp][kScoreU][H][E]
}

template <int SP, int G, int E, bool kHasM, bool kCheck>
__global__ void __launch_bounds__(kScoreThreads, 2) place_score_kernel(const ScoreParams p) {
    constexpr int kU = kScoreU;
    constexpr int H = G > 32 ? G / 32 : 1;              // table halves == ranks per lane
    constexpr int SEG = G < 32 ? G : 32, UPW = 32 / SEG;
    constexpr int NS = G * SP;
    constexpr int NW = (SP + 1) / 2;                    // words holding one rank's ids
    static_assert(SEG >= 4, "the joint reduction needs four lanes per unit");
    static_assert((E & (E - 1)) == 0 && E <= 256, "E");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const unsigned char* wc_b = smem_raw;                               // [H][E][32] float2
    const unsigned char* mu_b = smem_raw + (size_t)H * E * 256;         // [H][E][32] u32 (kHasM)
    const int l = blockIdx.y;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int sub = lane / SEG, g0 = lane % SEG;

    const int p_begin = blockIdx.x * p.chunk, p_end = min(p.P, p_begin + p.chunk);
    constexpr int kStride = (kScoreThreads / 32) * UPW;                 // candidates between two units of a warp pass
    const size_t stride_words = (size_t)kStride * p.L * NS / 2;
    int cand = p_begin + warp * UPW + sub;                              // unit 0 of this lane; unit u is cand + u * kStride
    const uint32_t* rowp = reinterpret_cast<const uint32_t*>(p.cand + ((size_t)cand * p.L + l) * NS);
    uint32_t bufA[kU][H][NW], bufB[kU][H][NW];
    auto fetch = [&](const uint32_t* row, uint32_t (&w)[H][NW]) {
#pragma unroll
        for (int rr = 0; rr < H; ++rr) {
            const int g = g0 + rr * 32;
            if constexpr (SP % 8 == 0) {
#pragma unroll
                for (int q = 0; q < SP / 8; ++q) {
                    const uint4 v = __ldcs(reinterpret_cast<const uint4*>(row + g * (SP / 2)) + q);
                    w[rr][4 * q] = v.x; w[rr][4 * q + 1] = v.y; w[rr][4 * q + 2] = v.z; w[rr][4 * q + 3] = v.w;
                }
            } else if constexpr (SP % 4 == 0) {
#pragma unroll
                for (int q = 0; q < SP / 4; ++q) {
                    const uint2 v = __ldcs(reinterpret_cast<const uint2*>(row + g * (SP / 2)) + q);
                    w[rr][2 * q] = v.x; w[rr][2 * q + 1] = v.y;
                }
            } else {
#pragma unroll
                for (int j = 0; j < NW; ++j) w[rr][j] = __ldcs(row + ((g * SP) >> 1) + j);
            }
        }
    };
    // the first rows are on their way while the table is staged
#pragma unroll
    for (int u = 0; u < kU; ++u)
        if (cand + u * kStride < p_end) fetch(rowp + u * stride_words, bufA[u]);
    {
        // all of a thread's table loads are in flight before the first store (the whole wave stages at once)
        constexpr int N4 = H * E * 16, kIt = (N4 + kScoreThreads - 1) / kScoreThreads;
        const uint4* src = reinterpret_cast<const uint4*>(p.t.wc + (size_t)l * H * E * 32);
        uint4* dst = reinterpret_cast<uint4*>(smem_raw);
        uint4 tmp[kIt];
#pragma unroll
        for (int k = 0; k < kIt; ++k)
            if ((int)threadIdx.x + k * kScoreThreads < N4) tmp[k] = __ldg(src + threadIdx.x + k * kScoreThreads);
#pragma unroll
        for (int k = 0; k < kIt; ++k)
            if ((int)threadIdx.x + k * kScoreThreads < N4) dst[threadIdx.x + k * kScoreThreads] = tmp[k];
        if constexpr (kHasM) {
            const uint4* ms = reinterpret_cast<const uint4*>(p.t.mu + (size_t)l * H * E * 32);
            uint4* md = reinterpret_cast<uint4*>(smem_raw + (size_t)H * E * 256);
            for (int i = threadIdx.x; i < H * E * 8; i += kScoreThreads) md[i] = ms[i];
        }
    }
    const uint32_t seg_mask = SEG == 32 ? 0xffffffffu : (((1u << SEG) - 1u) << (sub * SEG));
    const double sumB = p.t.sumB[l];
    const float sumB_hi = (float)sumB, sumB_lo = (float)(sumB - (double)sumB_hi);
    constexpr uint32_t emask2 = (uint32_t)(E - 1) | ((uint32_t)(E - 1) << 16);
    const uint32_t lane8 = (uint32_t)lane * 8u;         // table column of this lane's rank (replicated columns when G < 32)
    const float M_scalar = p.M_scalar;
    float4* const partial = p.partial;
    const int L = p.L;
    float mx0[kHasM ? H : 1][kHasM ? SP : 1];           // M of x0's own cells on this lane's rank(s)
    if constexpr (kHasM) {
#pragma unroll
        for (int rr = 0; rr < H; ++rr)
#pragma unroll
            for (int j = 0; j < SP; ++j) mx0[rr][j] = p.t.mx0[(size_t)l * NS + (g0 + rr * 32) * SP + j];
    }
    // kCheck: this unit's rank masks, one [H][E] array per candidate in flight; lane g0 reads back experts 4*(g0 + k*SEG) .. +3
    constexpr int EPL4 = E / SEG / 4;                    // 16-byte groups of experts per lane (1 or 2)
    static_assert(!kCheck || (E % (4 * SEG) == 0 && EPL4 >= 1 && EPL4 <= 2), "readback layout");
    uint32_t* mk_unit = reinterpret_cast<uint32_t*>(smem_raw + (size_t)H * E * (kHasM ? 384 : 256)) + (size_t)((warp * UPW + sub) * kU) * H * E;
    uint32_t r0p[kCheck ? EPL4 : 1];
    if constexpr (kCheck) {
        for (int i = threadIdx.x; i < (kScoreThreads / 32) * UPW * kU * H * E; i += kScoreThreads)
            reinterpret_cast<uint32_t*>(smem_raw + (size_t)H * E * (kHasM ? 384 : 256))[i] = 0u;
#pragma unroll
        for (int k = 0; k < EPL4; ++k) {
            const int32_t* r4 = p.t.r + (size_t)l * E + 4 * (g0 + k * SEG);
            r0p[k] = (uint32_t)min(r4[0], 255) | ((uint32_t)min(r4[1], 255) << 8) | ((uint32_t)min(r4[2], 255) << 16) | ((uint32_t)min(r4[3], 255) << 24);
        }
    }
    const uint32_t rank_bit = 1u << g0;
    __syncthreads();

    // one warp pass: prefetch the next pass into `nxt`, score the two candidates in `cur`, reduce, store
    auto pass = [&](uint32_t (&cur)[kU][H][NW], uint32_t (&nxt)[kU][H][NW]) {
        rowp += kU * stride_words;
#pragma unroll
        for (int u = 0; u < kU; ++u)
            if (cand + (kU + u) * kStride < p_end) fetch(rowp + u * stride_words, nxt[u]);
        float sq[kU], comm[kU], mig[kU], mx[kU];
        uint32_t kept[kU];
        uint32_t viol[kU], range[kU];
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            viol[u] = range[u] = 0u;
            // no activity test here: a unit past the end scores whatever its registers hold (ids are masked) and is not stored
            sq[u] = comm[u] = mig[u] = mx[u] = 0.0f;
            kept[u] = 0;
#pragma unroll
            for (int rr = 0; rr < H; ++rr) {
                uint32_t w[NW];
#pragma unroll
                for (int j = 0; j < NW; ++j) w[j] = cur[u][rr][j];
                if constexpr (SP % 2 == 1) {
                    // odd ranks start in the upper half of their first word: realign
                    const uint32_t sh = ((g0 + rr * 32) & 1) * 16;
#pragma unroll
                    for (int j = 0; j + 1 < NW; ++j) w[j] = __funnelshift_r(w[j], w[j + 1], sh);
                    w[NW - 1] = w[NW - 1] >> sh;
                }
                if constexpr (kCheck) {
#pragma unroll
                    for (int j = 0; j < NW; ++j) range[u] |= w[j];      // any bit outside an id's range marks the candidate invalid
                }
                if constexpr (E < 256) {                // E == 256: the PRMT below only takes the low byte of an id
#pragma unroll
                    for (int j = 0; j < NW; ++j) w[j] &= emask2;
                }
                float lg2[2] = {0.0f, 0.0f}, cm2[2] = {0.0f, 0.0f};  // two chains each: half the dependent adds
                uint32_t kp2[2] = {0u, 0u};
                uint32_t kbits = 0;
#pragma unroll
                for (int j = 0; j < SP; ++j) {
                    const uint32_t off = __byte_perm(w[j >> 1], lane8, (j & 1) ? 0x5524 : 0x5504);   // id << 8 | lane * 8
                    const float2 wc = *reinterpret_cast<const float2*>(wc_b + rr * E * 256 + off);
                    lg2[j & 1] += wc.x;
                    cm2[j & 1] += fabsf(wc.y);
                    if constexpr (kCheck)                   // x[e, rank] |= 1; the word that comes back says whether it was set already
                        viol[u] |= atomicOr(reinterpret_cast<uint32_t*>(reinterpret_cast<unsigned char*>(mk_unit + (u * H + rr) * E) + ((off >> 6) & 0x3fcu)), rank_bit);
                    if constexpr (kHasM) {
                        const uint32_t uw = *reinterpret_cast<const uint32_t*>(mu_b + rr * E * 128 + (off >> 1));
                        mig[u] += fmaxf(__uint_as_float(uw), 0.0f);                     // entering cell: + M
                        kbits |= (uint32_t)((int32_t)uw >> 31) & uw;                    // retained cell: which of x0's slots
                    } else {
                        kp2[j & 1] += __float_as_uint(wc.y) >> 31;
                    }
                }
                const float lg = lg2[0] + lg2[1];
                comm[u] += cm2[0] + cm2[1];
                kept[u] += kp2[0] + kp2[1];
                if constexpr (kHasM) {
#pragma unroll
                    for (int j = 0; j < SP; ++j) mig[u] += ((kbits >> j) & 1u) ? 0.0f : mx0[rr][j];   // leaving cells, x0's slot order
                }
                const float d = __fsub_rn(__fmaf_rn(lg, (float)G, -sumB_hi), sumB_lo);   // G*L_g - sum_g L_g
                sq[u] = __fmaf_rn(d, d, sq[u]);
                mx[u] = fmaxf(mx[u], lg);
            }
        }
        bool bad0 = false, bad1 = false, same0 = true, same1 = true;
        if constexpr (kCheck) {
            __syncwarp();
#pragma unroll
            for (int u = 0; u < kU; ++u) {
                bool same = true, missing = false;
#pragma unroll
                for (int k = 0; k < EPL4; ++k) {
                    uint32_t cnt = 0;
#pragma unroll
                    for (int rr = 0; rr < H; ++rr) {
                        uint4* q = reinterpret_cast<uint4*>(mk_unit + (u * H + rr) * E) + g0 + k * SEG;
                        const uint4 a = *q;
                        *q = make_uint4(0u, 0u, 0u, 0u);
                        cnt += __popc(a.x) | (__popc(a.y) << 8) | (__popc(a.z) << 16) | (__popc(a.w) << 24);
                    }
                    same = same && cnt == r0p[k];
                    missing = missing || ((~(((cnt & 0x7f7f7f7fu) + 0x7f7f7f7fu) | cnt) & 0x80808080u) != 0u);
                }
                const bool bad_l = ((viol[u] & rank_bit) != 0u) || ((range[u] & ~emask2) != 0u) || missing;
                const uint32_t bb = __ballot_sync(0xffffffffu, bad_l) & seg_mask, ss = __ballot_sync(0xffffffffu, !same) & seg_mask;
                if (u == 0) { bad0 = bb != 0u; same0 = ss == 0u; } else { bad1 = bb != 0u; same1 = ss == 0u; }
            }
            __syncwarp();                                   // the masks are clear before the next pass ORs into them
        }
        // one transposed butterfly for both candidates of the unit: after the first step the lanes with bit h clear
        // work for candidate 0 and the others for candidate 1, after the second the lanes with bit h2 clear hold sq, the
        // others comm
        constexpr int h = SEG >> 1, h2 = SEG >> 2;
        const bool up = (lane & h) != 0, up2 = (lane & h2) != 0;
        float ka = (up ? sq[1] : sq[0]) + __shfl_xor_sync(0xffffffffu, up ? sq[0] : sq[1], h);
        float kb = (up ? comm[1] : comm[0]) + __shfl_xor_sync(0xffffffffu, up ? comm[0] : comm[1], h);
        float v = (up2 ? kb : ka) + __shfl_xor_sync(0xffffffffu, up2 ? ka : kb, h2);
#pragma unroll
        for (int o = h2 >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        const float commt = __shfl_xor_sync(0xffffffffu, v, h2);            // lanes with bit h2 clear: v = sq, commt = comm
        const float mxa0 = __uint_as_float(__reduce_max_sync(seg_mask, __float_as_uint(mx[0])));   // loads are >= 0
        const float mxa1 = __uint_as_float(__reduce_max_sync(seg_mask, __float_as_uint(mx[1])));
        float migt;
        if constexpr (kHasM) {
            float m = (up ? mig[1] : mig[0]) + __shfl_xor_sync(0xffffffffu, up ? mig[0] : mig[1], h);
#pragma unroll
            for (int o = h >> 1; o > 0; o >>= 1) m += __shfl_xor_sync(0xffffffffu, m, o);
            migt = m;
        } else {
            const uint32_t k2 = __reduce_add_sync(seg_mask, kept[0] | (kept[1] << 16));       // each total <= NS < 2^16
            const int k = up ? (int)(k2 >> 16) : (int)(k2 & 0xffffu);
            migt = M_scalar * (float)(2 * (NS - k));                                          // entering + leaving cells, M each: exact
        }
        // lane g0 == 0 writes candidate 0, lane g0 == h candidate 1
        const int mine = cand + (up ? kStride : 0);
        if ((g0 & (h - 1)) == 0 && mine < p_end) {
            float4 res = make_float4(v, commt, migt, up ? mxa1 : mxa0);
            if constexpr (kCheck) {
                const bool bad = up ? bad1 : bad0, same = up ? same1 : same0;
                if (bad) res = make_float4(CUDART_NAN_F, CUDART_NAN_F, CUDART_NAN_F, CUDART_NAN_F);
                p.status[(size_t)l * p.P + mine] = bad ? 1 : ((!same || p.force_general) ? 2 : 0);
            }
            partial[(size_t)mine * L + l] = res;
        }
        cand += kU * kStride;
    };
    for (int pc = p_begin + warp * UPW; pc < p_end; pc += 2 * kU * kStride) {
        pass(bufA, bufB);
        if (pc + kU * kStride >= p_end) break;
        pass(bufB, bufA);
    }
}

// The 9-slots-per-rank shape (32 ranks, 288 slots, 256 experts; scalar M, no fused validation) with the candidate rows
// delivered by TMA.  A rank's 18 bytes start on an odd half-word for every other rank, so the per-lane global loads of
// place_score_kernel touch all 18 sectors of a row in each of their five instructions (92 tag look-ups per row); here ONE
// tiled copy per warp pass brings two rows into the warp's shared-memory ring.  The tensor map sees a row as 4 pieces of
// 72 ids and asks for a box 80 ids wide: each piece lands at a 160-byte pitch (tail zero-filled), which spreads the 32
// lanes' words over the 32 banks -- five conflict-free LDS.32 per lane and row.  No L1 tag traffic, no register ping-pong.
constexpr int kTmaRowPitch = 640;                     // 4 pieces x 160 B
constexpr int kTmaSlots = 2;                          // ring slots per warp, one pass (two rows) each
inline size_t place_score_tma_smem_bytes() {
    // table + per-warp ring + per-warp (full, empty) barrier of every slot
    return (size_t)256 * 256 + (size_t)(kScoreThreads / 32) * kTmaSlots * kScoreU * kTmaRowPitch + (kScoreThreads / 32) * kTmaSlots * 16;
}

__device__ __forceinline__ uint32_t lds_u32_ordered(uint32_t addr) {      // ordered among the volatile asm statements (barrier wait before, refill after)
    uint32_t v;
    asm volatile("ld.shared.b32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ float2 lds_f32x2(uint32_t addr) {               // a table cell; its address depends on words read after the barrier wait
    float2 v;
    asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}

// How a warp hands a ring slot it has read back to the copy engine (see the comment at the refill): 0 = the copy's coordinate
// depends on every word the warp loaded (default, the only variant that is both correct and free), 1 = release / acquire on an
// "empty" mbarrier, 2 = fence.proxy.async.  1 and 2 exist for the record in profiles/r3_k4_tma_handoff.md.
#ifndef GIMBAL_TMA_HANDOFF
#define GIMBAL_TMA_HANDOFF 0
#endif
__global__ void __launch_bounds__(kScoreThreads, 2) place_score_tma_kernel(const ScoreParams p, const __grid_constant__ CUtensorMap tm) {
    constexpr int SP = 9, G = 32, E = 256, NS = G * SP, NW = 5, kU = kScoreU, kWarps = kScoreThreads / 32;
    constexpr uint32_t kPassBytes = kU * kTmaRowPitch;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const int l = blockIdx.y;
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);          // warp-uniform for the compiler too
    const int lane = threadIdx.x & 31;
    const int p_begin = blockIdx.x * p.chunk, p_end = min(p.P, p_begin + p.chunk);
    constexpr int kPassStride = kWarps * kU;                                         // candidates between two passes of a warp
    const int c_first = p_begin + warp * kU;
    const uint32_t tab_a = __shfl_sync(0xffffffffu, ptx::smem_u32(smem_raw), 0);     // [E][32] float2
    const uint32_t ring_a = tab_a + (uint32_t)E * 256u + (uint32_t)warp * (kTmaSlots * kPassBytes);          // [slots][kU][640] of this warp
    // this warp's barriers: "full" of slot s at bar_a + 8 s (the copy's bytes have landed); the "empty" barriers behind them are
    // only used by the GIMBAL_TMA_HANDOFF == 1 build
    const uint32_t bar_a = tab_a + (uint32_t)E * 256u + (uint32_t)kWarps * (kTmaSlots * kPassBytes) + (uint32_t)warp * (kTmaSlots * 16);
    constexpr uint32_t kEmptyOff = kTmaSlots * 8;
    const uint64_t pol = ptx::policy_evict_first();
    if (ptx::elect_one()) {
#pragma unroll
        for (int s = 0; s < kTmaSlots; ++s) { ptx::mbar_init(bar_a + 8 * s, 1); ptx::mbar_init(bar_a + kEmptyOff + 8 * s, 1); }
        ptx::fence_barrier_init();
        ptx::fence_proxy_async();
        // the first rows are on their way while the table is staged
#pragma unroll
        for (int s = 0; s < kTmaSlots; ++s) {
            const int c = c_first + s * kPassStride;
            if (c < p_end) {
                ptx::mbar_arrive_expect_tx(bar_a + 8 * s, kPassBytes);
                ptx::tma_load_4d(ring_a + s * kPassBytes, &tm, bar_a + 8 * s, 0, 0, l, c, pol);
            }
        }
    }
    {
        // the table {w, c}[E][32] is put together from its compact halves: c[E][32] and w[E] (half the bytes out of L2); a thread
        // takes two cells at a time, so a warp's 16-byte stores are contiguous (no bank conflicts)
        constexpr int N2 = E * 16, kIt = N2 / kScoreThreads;
        const float2* src = reinterpret_cast<const float2*>(p.t.c_s + (size_t)l * E * 32);
        const float* wsrc = p.t.w_f + (size_t)l * E;
        float4* dst = reinterpret_cast<float4*>(smem_raw);
        float2 tmp[kIt];
        float wv[kIt];
#pragma unroll
        for (int k = 0; k < kIt; ++k) {
            tmp[k] = __ldg(src + threadIdx.x + k * kScoreThreads);
            wv[k] = __ldg(wsrc + ((threadIdx.x + k * kScoreThreads) >> 4));
        }
#pragma unroll
        for (int k = 0; k < kIt; ++k) dst[threadIdx.x + k * kScoreThreads] = make_float4(wv[k], tmp[k].x, wv[k], tmp[k].y);
    }
    const double sumB = p.t.sumB[l];
    const float sumB_hi = (float)sumB, sumB_lo = (float)(sumB - (double)sumB_hi);
    const uint32_t lane8 = (uint32_t)lane * 8u;
    const float M_scalar = p.M_scalar;
    float4* const partial = p.partial;
    const int L = p.L;
    // this lane's rank: piece lane / 8, then 18 bytes per rank inside the piece (word-aligned start, odd ranks begin in the upper half)
    const uint32_t lane_off = (uint32_t)(lane >> 3) * 160u + 4u * ((9u * (uint32_t)(lane & 7)) >> 1);
    const uint32_t sh = (uint32_t)(lane & 1) * 16u;
    __syncthreads();

    // one warp pass: two rows out of the ring, scored into slots `q`, `q + 1` of the pending results
    float sq[2 * kU], comm[2 * kU], mx[2 * kU];
    uint32_t kept[2 * kU];
    uint32_t it = 0;
    auto pass = [&](int c0, int q) {
        const uint32_t slot = it & (kTmaSlots - 1), phase = (it / kTmaSlots) & 1u;
        const uint32_t bar = bar_a + 8 * slot, rows = ring_a + slot * kPassBytes;
        ptx::mbar_wait(bar, phase);
        ++it;
        uint32_t w[kU][NW];
#pragma unroll
        for (int u = 0; u < kU; ++u)
#pragma unroll
            for (int j = 0; j < NW; ++j) w[u][j] = lds_u32_ordered(rows + u * kTmaRowPitch + 4 * j + lane_off);
        // refill the slot with the pass after next.  The copy (async proxy) overwrites what the loads above read, and it must not
        // start before every lane's loads have RETURNED: at kernel start, when all warps of an SM fire at once behind the table's
        // stores, queued loads lose that race.  Measured on the bench grid (4096 candidates x 58 layers, 300 launches,
        // profiles/r3_k4_tma_handoff.md): the textbook hand-off -- arrive on an "empty" mbarrier after the loads, wait on it, then
        // expect_tx + copy -- still returned wrong rows in 14 launches (the barrier unit is not ordered behind the warp's queued
        // shared-memory loads, and nothing waits for their scoreboard); fence.proxy.async before the copy was correct but 2 us
        // slower.  What holds by construction, at no cost: the copy's candidate coordinate carries a true dependency on ALL ten
        // words of every lane (warp OR-reduction, AND-ed with a kernel argument that is 0 at run time and that the compiler
        // cannot fold), so UTMALDG cannot issue before the last load has delivered its register.
        if (c0 + kTmaSlots * kPassStride < p_end) {
#if GIMBAL_TMA_HANDOFF == 0
            uint32_t acc = 0u;
#pragma unroll
            for (int u = 0; u < kU; ++u)
#pragma unroll
                for (int j = 0; j < NW; ++j) acc |= w[u][j];
            const uint32_t dep = __reduce_or_sync(0xffffffffu, acc & p.zero);
            if (ptx::elect_one()) {
                ptx::mbar_arrive_expect_tx(bar, kPassBytes);
                ptx::tma_load_4d(rows, &tm, bar, 0, 0, l, c0 + kTmaSlots * kPassStride + (int)dep, pol);
            }
#else
            __syncwarp();
            if (ptx::elect_one()) {
#if GIMBAL_TMA_HANDOFF == 1
                ptx::mbar_arrive(bar + kEmptyOff);          // the slot's k-th refill completes phase k: same parity as the full barrier
                ptx::mbar_wait(bar + kEmptyOff, phase);
#else
                ptx::fence_proxy_async();
#endif
                ptx::mbar_arrive_expect_tx(bar, kPassBytes);
                ptx::tma_load_4d(rows, &tm, bar, 0, 0, l, c0 + kTmaSlots * kPassStride, pol);
            }
#endif
        }
#pragma unroll
        for (int u = 0; u < kU; ++u) {
#pragma unroll
            for (int j = 0; j + 1 < NW; ++j) w[u][j] = __funnelshift_r(w[u][j], w[u][j + 1], sh);
            w[u][NW - 1] = w[u][NW - 1] >> sh;
            float lg2[2], cm2[2];
            uint32_t kp2[2];
#pragma unroll
            for (int j = 0; j < SP; ++j) {
                const uint32_t off = __byte_perm(w[u][j >> 1], lane8, (j & 1) ? 0x5524 : 0x5504);   // id << 8 | lane * 8
                const float2 wc = lds_f32x2(tab_a + off);
                if (j < 2) {
                    lg2[j] = wc.x; cm2[j] = fabsf(wc.y); kp2[j] = __float_as_uint(wc.y) >> 31;
                } else {
                    lg2[j & 1] += wc.x;
                    cm2[j & 1] += fabsf(wc.y);
                    kp2[j & 1] += __float_as_uint(wc.y) >> 31;
                }
            }
            const float lg = lg2[0] + lg2[1];
            comm[q + u] = cm2[0] + cm2[1];
            kept[q + u] = kp2[0] + kp2[1];
            const float d = __fsub_rn(__fmaf_rn(lg, (float)G, -sumB_hi), sumB_lo);   // G*L_g - sum_g L_g
            sq[q + u] = d * d;
            mx[q + u] = lg;
        }
    };
    // Two passes share one transposed butterfly over their four rows (eight sums): lane bits 16 and 8 pick the row, bit 4 the
    // kind (sq / comm) -- 4 + 2 + 1 + 1 + 1 shuffles and one exchange for four rows.  Row r = (bit16, bit8) is candidate
    // c0 + (r & 1) of pass r >> 1.
    const bool b16 = (lane & 16) != 0, b8 = (lane & 8) != 0, b4 = (lane & 4) != 0;
    for (int c0 = c_first; c0 < p_end; c0 += 2 * kPassStride) {
        pass(c0, 0);
        const bool two = c0 + kPassStride < p_end;
        if (two) pass(c0 + kPassStride, kU);
        else {
#pragma unroll
            for (int u = 0; u < kU; ++u) sq[kU + u] = comm[kU + u] = mx[kU + u] = 0.0f, kept[kU + u] = 0u;
        }
        float s0 = (b16 ? sq[2] : sq[0]) + __shfl_xor_sync(0xffffffffu, b16 ? sq[0] : sq[2], 16);
        float s1 = (b16 ? sq[3] : sq[1]) + __shfl_xor_sync(0xffffffffu, b16 ? sq[1] : sq[3], 16);
        float m0 = (b16 ? comm[2] : comm[0]) + __shfl_xor_sync(0xffffffffu, b16 ? comm[0] : comm[2], 16);
        float m1 = (b16 ? comm[3] : comm[1]) + __shfl_xor_sync(0xffffffffu, b16 ? comm[1] : comm[3], 16);
        const float s = (b8 ? s1 : s0) + __shfl_xor_sync(0xffffffffu, b8 ? s0 : s1, 8);
        const float m = (b8 ? m1 : m0) + __shfl_xor_sync(0xffffffffu, b8 ? m0 : m1, 8);
        float v = (b4 ? m : s) + __shfl_xor_sync(0xffffffffu, b4 ? s : m, 4);
        v += __shfl_xor_sync(0xffffffffu, v, 2);
        v += __shfl_xor_sync(0xffffffffu, v, 1);
        const float commt = __shfl_xor_sync(0xffffffffu, v, 4);                 // lanes with bit 4 clear: v = sq, commt = comm
        const float mxa0 = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(mx[0])));   // loads are >= 0
        const float mxa1 = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(mx[1])));
        const float mxa2 = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(mx[2])));
        const float mxa3 = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(mx[3])));
        const uint32_t k01 = __reduce_add_sync(0xffffffffu, kept[0] | (kept[1] << 16));
        const uint32_t k23 = __reduce_add_sync(0xffffffffu, kept[2] | (kept[3] << 16));
        const uint32_t kk = b16 ? k23 : k01;
        const int k = b8 ? (int)(kk >> 16) : (int)(kk & 0xffffu);
        const float migt = M_scalar * (float)(2 * (NS - k));
        const float mxa = b16 ? (b8 ? mxa3 : mxa2) : (b8 ? mxa1 : mxa0);
        const int mine = c0 + (b16 ? kPassStride : 0) + (b8 ? 1 : 0);
        if ((lane & 7) == 0 && mine < p_end) partial[(size_t)mine * L + l] = make_float4(v, commt, migt, mxa);
    }
}

// Same contract for any supported shape (runtime slots per rank <= 16, G a power of two <= 64, any E <= 256):
// scalar loads, ids clamped to the table.
template <bool kHasM>
__global__ void __launch_bounds__(kScoreThreads, 1) place_score_generic_kernel(const ScoreParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int GP = place_gp(p.G), H = GP / 32, E = p.E, sp = p.sp, NS = p.G * p.sp;
    const float2* wc_s = reinterpret_cast<const float2*>(smem_raw);                       // [H][E][32]
    const uint32_t* mu_s = reinterpret_cast<const uint32_t*>(smem_raw + (size_t)H * E * 256);
    const int l = blockIdx.y;
    {
        const uint4* src = reinterpret_cast<const uint4*>(p.t.wc + (size_t)l * H * E * 32);
        uint4* dst = reinterpret_cast<uint4*>(smem_raw);
        for (int i = threadIdx.x; i < H * E * 16; i += kScoreThreads) dst[i] = src[i];
        if constexpr (kHasM) {
            const uint4* ms = reinterpret_cast<const uint4*>(p.t.mu + (size_t)l * H * E * 32);
            uint4* md = reinterpret_cast<uint4*>(smem_raw + (size_t)H * E * 256);
            for (int i = threadIdx.x; i < H * E * 8; i += kScoreThreads) md[i] = ms[i];
        }
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int seg = p.G < 32 ? p.G : 32, upw = 32 / seg;
    const int sub = lane / seg, g0 = lane % seg;
    const double Gd = (double)p.G, sumB = p.t.sumB[l];
    const uint32_t emax = (uint32_t)E - 1u;
    const int p_begin = blockIdx.x * p.chunk, p_end = min(p.P, p_begin + p.chunk);
    const int stride = (kScoreThreads / 32) * upw;
    for (int pc = p_begin + warp * upw; pc < p_end; pc += stride) {
        const int cand = pc + sub;
        const bool active = cand < p_end;
        float sq = 0.0f, comm = 0.0f, mig = 0.0f, mx = 0.0f;
        int kept = 0;
        if (active) {
            const int16_t* row = p.cand + ((size_t)cand * p.L + l) * NS;
            for (int rr = 0; rr < H; ++rr) {
                const int g = g0 + rr * 32;
                float lg = 0.0f;
                uint32_t kbits = 0;
                for (int j = 0; j < sp; ++j) {
                    const uint32_t x = min((uint32_t)(uint16_t)__ldcs(row + g * sp + j), emax);
                    const int idx = (rr * E + (int)x) * 32 + lane;
                    const float2 wc = wc_s[idx];
                    lg += wc.x;
                    comm += fabsf(wc.y);
                    if constexpr (kHasM) {
                        const uint32_t u = mu_s[idx];
                        mig += fmaxf(__uint_as_float(u), 0.0f);
                        kbits |= (uint32_t)((int32_t)u >> 31) & u;
                    } else {
                        kept += (int)(__float_as_uint(wc.y) >> 31);
                    }
                }
                if constexpr (kHasM) {
                    for (int j = 0; j < sp; ++j) mig += ((kbits >> j) & 1u) ? 0.0f : p.t.mx0[(size_t)l * NS + g * sp + j];
                }
                const float d = (float)((double)lg * Gd - sumB);
                sq = __fmaf_rn(d, d, sq);
                mx = fmaxf(mx, lg);
            }
        }
        // butterflies over the seg lanes of the unit (xor offsets below seg stay inside it)
        for (int o = seg >> 1; o > 0; o >>= 1) {
            sq += __shfl_xor_sync(0xffffffffu, sq, o);
            comm += __shfl_xor_sync(0xffffffffu, comm, o);
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
            if constexpr (kHasM) mig += __shfl_xor_sync(0xffffffffu, mig, o);
            else kept += __shfl_xor_sync(0xffffffffu, kept, o);
        }
        if constexpr (!kHasM) mig = p.M_scalar * (float)(2 * (NS - kept));
        if (active && g0 == 0) p.partial[(size_t)cand * p.L + l] = make_float4(sq, comm, mig, mx);
    }
}

// ------------------------------------------------------------------------------------------
// Exact validation, and the plain definition for candidates whose replica counts differ from x0's.
// ------------------------------------------------------------------------------------------
struct CheckParams {
    int P, L, E, G, sp, chunk;
    int force_general;                  // tests: score every valid candidate here
    float M_scalar;
    const int16_t* cand;                // [P,L,NS]
    const int16_t* prev;                // [L,NS]
    const float* M;                     // caller's [L,E,G] | nullptr
    PlaceTables t;
    float4* partial;
    uint8_t* status;                    // [L,P] 0: valid, same copies as x0   1: invalid   2: valid, other replica counts
};

constexpr int kCheckWarps = 8;
constexpr int kCheckE = 256;            // rank-mask rows per half (E <= 256, ids are masked to 8 bits)

inline size_t place_check_smem_bytes(int G) { return sizeof(uint32_t) * (size_t)kCheckWarps * (G > 32 ? 2 : 1) * kCheckE + 2 * kCheckE; }

// the candidate's own score (PAPER.md:236-248 with r from the candidate, R12); lane <-> rank, global tables.
// mk: the warp's rank masks [H][256] of this candidate.
__device__ __forceinline__ void place_score_own_r(const CheckParams& p, int l, int c, const int16_t* row, const uint32_t* mk, int lane) {
    const int E = p.E, NS = p.G * p.sp, H = p.G > 32 ? 2 : 1;
    const double Gd = (double)p.G, sumB = p.t.sumB[l];
    float sq = 0.0f, comm = 0.0f, mig = 0.0f, mx = 0.0f;
    const int16_t* pv = p.prev + (size_t)l * NS;
    for (int rr = 0; rr < H; ++rr) {
        const int g = lane + rr * 32;
        if (g >= p.G) break;
        double lgd = 0.0;
        for (int j = 0; j < p.sp; ++j) {
            const int e = row[g * p.sp + j];
            const int r = __popc(mk[e]) + (H == 2 ? __popc(mk[kCheckE + e]) : 0);
            lgd += p.t.b_raw[(size_t)l * E + e] / (double)r;
            comm += p.t.c_raw[((size_t)l * E + e) * p.G + g] / (float)r;
            if (!((p.t.pmask[(size_t)l * E + e] >> g) & 1ull))                 // cell enters
                mig += p.M ? p.M[((size_t)l * E + e) * p.G + g] : p.M_scalar;
            const int e0 = pv[g * p.sp + j];
            if (!((mk[(g >> 5) * kCheckE + e0] >> (g & 31)) & 1u))             // x0's cell leaves
                mig += p.M ? p.M[((size_t)l * E + e0) * p.G + g] : p.M_scalar;
        }
        const float d = (float)(lgd * Gd - sumB);
        sq = __fmaf_rn(d, d, sq);
        mx = fmaxf(mx, (float)lgd);
    }
    for (int o = 16; o > 0; o >>= 1) {
        sq += __shfl_xor_sync(0xffffffffu, sq, o);
        comm += __shfl_xor_sync(0xffffffffu, comm, o);
        mig += __shfl_xor_sync(0xffffffffu, mig, o);
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if (lane == 0) p.partial[(size_t)c * p.L + l] = make_float4(sq, comm, mig, mx);
}

// grid (chunks, L), kCheckWarps warps; a warp takes one (candidate, layer) at a time, lane <-> rank (two ranks per
// lane when G = 64).  SP: compile-time slots per rank (0: runtime, up to 16).
//   scatter   every slot ORs its rank's bit into the candidate's x[e, .] row: mk[e] |= 1 << g.  The word that comes
//             back tells whether the bit was already there ("twice on one rank"); ids are masked to 8 bits, the range
//             check is one OR over the packed words (plus a compare per slot when E is not a power of two).
//   readback  lane i owns experts 4i..4i+3 and 128+4i..: two 16-byte loads return its eight rank masks, two 16-byte
//             stores clear them for the next candidate; their popcounts, packed four to a word, are compared with x0's
//             replica counts in one XOR each.  All equal <=> same copies as x0 (place_score_kernel's premise).
template <int SP, int H>
__global__ void __launch_bounds__(kCheckWarps * 32) place_check_kernel(const CheckParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int E = p.E, sp = SP > 0 ? SP : p.sp, NS = p.G * sp;
    uint32_t* mk_all = reinterpret_cast<uint32_t*>(smem_raw);                                 // [warps][H][256] rank masks
    uint8_t* r0_s = reinterpret_cast<uint8_t*>(mk_all + kCheckWarps * H * kCheckE);           // [256] replica counts of x0 (0 past E)
    const int l = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int e = threadIdx.x; e < kCheckE; e += kCheckWarps * 32) r0_s[e] = e < E ? (uint8_t)min(p.t.r[(size_t)l * E + e], 255) : 0;
    for (int i = threadIdx.x; i < kCheckWarps * H * kCheckE; i += kCheckWarps * 32) mk_all[i] = 0u;
    __syncthreads();
    uint32_t* mk = mk_all + warp * H * kCheckE;
    const uint32_t r0a = reinterpret_cast<const uint32_t*>(r0_s)[lane], r0b = reinterpret_cast<const uint32_t*>(r0_s)[32 + lane];
    const bool pow2E = (E & (E - 1)) == 0;
    const uint32_t id_ok = pow2E ? (uint32_t)(E - 1) : 0xffu;                                  // bits a valid id may use
    const uint32_t bit = 1u << lane;
    constexpr int MAXSP = SP > 0 ? SP : 16, NWL = MAXSP / 2 + 1;                              // words that can hold a rank's ids
    const int p_begin = blockIdx.x * p.chunk, p_end = min(p.P, p_begin + p.chunk);
    // this lane's ranks: where their ids start in a row (word, half-word shift) and how many words they span
    int w0[H], nw[H];
    uint32_t sh[H];
#pragma unroll
    for (int rr = 0; rr < H; ++rr) {
        const int hw0 = (lane + rr * 32) * sp;
        w0[rr] = hw0 >> 1; sh[rr] = (hw0 & 1) * 16; nw[rr] = (lane + rr * 32 < p.G) ? (sp + (hw0 & 1) + 1) >> 1 : 0;
    }
    uint32_t Wn[H][NWL];                                                                       // the next candidate's words
    auto fetch = [&](int c) {
        const uint32_t* roww = reinterpret_cast<const uint32_t*>(p.cand + ((size_t)c * p.L + l) * NS);
#pragma unroll
        for (int rr = 0; rr < H; ++rr)
#pragma unroll
            for (int k = 0; k < NWL; ++k) Wn[rr][k] = k < nw[rr] ? __ldcs(roww + w0[rr] + k) : 0u;
    };
    if (p_begin + warp < p_end) fetch(p_begin + warp);
    for (int c = p_begin + warp; c < p_end; c += kCheckWarps) {
        const int16_t* row = p.cand + ((size_t)c * p.L + l) * NS;
        uint32_t W[H][NWL + 1];
#pragma unroll
        for (int rr = 0; rr < H; ++rr) {
#pragma unroll
            for (int k = 0; k < NWL; ++k) W[rr][k] = Wn[rr][k];
            W[rr][NWL] = 0u;
        }
        if (c + kCheckWarps < p_end) fetch(c + kCheckWarps);                                   // in flight during this candidate
        uint32_t viol = 0, range = 0;
        bool oob = false;
#pragma unroll
        for (int rr = 0; rr < H; ++rr) {
            if (nw[rr] > 0) {
#pragma unroll
                for (int k = 0; k < NWL; ++k) W[rr][k] = __funnelshift_r(W[rr][k], W[rr][k + 1], sh[rr]);   // slot j of the rank = halfword j
                uint32_t* mkr = mk + rr * kCheckE;
#pragma unroll
                for (int j = 0; j < MAXSP; ++j) {
                    if (SP > 0 || j < sp) {
                        const uint32_t wj = W[rr][j >> 1];
                        const uint32_t raw = (j & 1) ? (wj >> 16) : (wj & 0xffffu);
                        range |= raw;
                        if (!pow2E) oob |= raw >= (uint32_t)E;
                        viol |= atomicOr(mkr + (raw & 255u), bit);
                    }
                }
            }
        }
        __syncwarp();
        // readback + clear
        uint32_t diff = 0, zero = 0;
#pragma unroll
        for (int rr = 0; rr < H; ++rr) {
            {
                uint4* q = reinterpret_cast<uint4*>(mk + rr * kCheckE);
                const uint4 a = q[lane], b = q[32 + lane];
                q[lane] = make_uint4(0u, 0u, 0u, 0u);
                q[32 + lane] = make_uint4(0u, 0u, 0u, 0u);
                const uint32_t ca = __popc(a.x) | (__popc(a.y) << 8) | (__popc(a.z) << 16) | (__popc(a.w) << 24);
                const uint32_t cb = __popc(b.x) | (__popc(b.y) << 8) | (__popc(b.z) << 16) | (__popc(b.w) << 24);
                if (rr == 0) { diff = ca; zero = cb; } else { diff += ca; zero += cb; }        // packed counts (each <= 64)
            }
        }
        const uint32_t cnta = diff, cntb = zero;
        const bool same = (cnta == r0a) && (cntb == r0b);
        // an expert of [0,E) hosted nowhere: a zero byte where x0's count is not zero (x0 valid: r0 >= 1 below E)
        const uint32_t za = ~(((cnta & 0x7f7f7f7fu) + 0x7f7f7f7fu) | cnta) & 0x80808080u, zb = ~(((cntb & 0x7f7f7f7fu) + 0x7f7f7f7fu) | cntb) & 0x80808080u;
        const uint32_t na = ~(((r0a & 0x7f7f7f7fu) + 0x7f7f7f7fu) | r0a) & 0x80808080u, nb = ~(((r0b & 0x7f7f7f7fu) + 0x7f7f7f7fu) | r0b) & 0x80808080u;
        const bool missing = ((za & ~na) | (zb & ~nb)) != 0;
        const bool bad_lane = ((viol & bit) != 0) || ((range & ~id_ok) != 0) || oob || missing;
        const bool bad = __any_sync(0xffffffffu, bad_lane);
        const bool all_same = __all_sync(0xffffffffu, same);
        if (lane == 0) {
            if (bad) p.partial[(size_t)c * p.L + l] = make_float4(CUDART_NAN_F, CUDART_NAN_F, CUDART_NAN_F, CUDART_NAN_F);
            p.status[(size_t)l * p.P + c] = bad ? 1 : ((!all_same || p.force_general) ? 2 : 0);
        }
        __syncwarp();
    }
}

// The candidates place_check_kernel marked "valid, other replica counts than x0" (status 2): rebuild the rank masks and
// score with the candidate's own r.  Same grid as the check; warps skip everything else.
__global__ void __launch_bounds__(kCheckWarps * 32) place_own_r_kernel(const CheckParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int NS = p.G * p.sp, H = p.G > 32 ? 2 : 1;
    uint32_t* mk_all = reinterpret_cast<uint32_t*>(smem_raw);
    const int l = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t* mk = mk_all + warp * H * kCheckE;
    for (int i = lane; i < H * kCheckE; i += 32) mk[i] = 0u;
    __syncwarp();
    const int p_begin = blockIdx.x * p.chunk, p_end = min(p.P, p_begin + p.chunk);
    // most calls have nothing to do here: the block reads its verdicts in one go and leaves
    int mine = 0;
    for (int c = p_begin + threadIdx.x; c < p_end; c += kCheckWarps * 32) mine |= p.status[(size_t)l * p.P + c] == 2;
    if (!__syncthreads_or(mine)) return;
    for (int c = p_begin + warp; c < p_end; c += kCheckWarps) {
        if (p.status[(size_t)l * p.P + c] != 2) continue;
        const int16_t* row = p.cand + ((size_t)c * p.L + l) * NS;
        for (int rr = 0; rr < H; ++rr) {
            const int g = lane + rr * 32;
            if (g < p.G)
                for (int j = 0; j < p.sp; ++j) atomicOr(mk + rr * kCheckE + (uint16_t)row[g * p.sp + j], 1u << lane);
        }
        __syncwarp();
        place_score_own_r(p, l, c, row, mk, lane);
        __syncwarp();
        for (int i = lane; i < H * kCheckE; i += 32) mk[i] = 0u;
        __syncwarp();
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

// a warp per candidate: lanes take the layers in strides of 32, fixed-shape tree over the lanes (deterministic), in double
__global__ void __launch_bounds__(256) place_finalize_kernel(const FinalizeParams p) {
    const int c = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    unsigned long long key = ~0ull;
    if (c < p.P) {
        double sq = 0.0, comm = 0.0, mig = 0.0, mx = 0.0;
        bool bad = *p.bad_prev != 0;
        for (int l = lane; l < p.L; l += 32) {
            const float4 v = p.partial[(size_t)c * p.L + l];
            if (v.x != v.x) bad = true;
            sq += v.x; comm += v.y; mig += v.z; mx += v.w;
        }
        for (int o = 16; o > 0; o >>= 1) {
            sq += __shfl_xor_sync(0xffffffffu, sq, o);
            comm += __shfl_xor_sync(0xffffffffu, comm, o);
            mig += __shfl_xor_sync(0xffffffffu, mig, o);
            mx += __shfl_xor_sync(0xffffffffu, mx, o);
        }
        bad = __any_sync(0xffffffffu, bad);
        const double load = sq / ((double)p.G * (double)p.G);
        float* o = p.out + (size_t)c * 5;
        const float J = (float)((double)p.alpha * comm + (double)p.beta * load + (double)p.gamma * mig);
        if (lane < 5) {
            const float vals[5] = {J, (float)load, (float)comm, (float)mig, (float)mx};
            o[lane] = bad ? CUDART_NAN_F : vals[lane];
        }
        if (!bad) key = ((unsigned long long)ordered_u32(J + 0.0f) << 32) | (unsigned)c;
    }
    if (p.best && lane == 0 && key != ~0ull) atomicMin(p.best, key);
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
    // per-slot rows of `cur` for the all-pairs kernel (move_slots_kernel)
    float* slotC;       // [L][NS][G]  c (sign = x0 hosts it) of the slot's expert on every rank
    float* slotM;       // [L][NS][G]  M of the slot's expert on every rank (M table only)
    double* slot_w;     // [L][NS]     load share of the slot's expert
    double* slot_u;     // [L][NS]     load of the slot's rank minus that share
    uint64_t* slot_cm;  // [L][NS]     ranks hosting the slot's expert in cur
    int2* slot_eg;      // [L][NS]     {expert, rank} of the slot
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
                const size_t i11 = tab_idx(p.E, e1, g1), i12 = tab_idx(p.E, e1, g2), i21 = tab_idx(p.E, e2, g1), i22 = tab_idx(p.E, e2, g2);
                const float2 t11 = wc[i11], t12 = wc[i12], t21 = wc[i21], t22 = wc[i22];
                // loads in double: L1 - L2 and w2 - w1 subtract nearly equal numbers that can exceed 2^24
                const double w1 = p.t.w_e[(size_t)l * p.E + e1], w2 = p.t.w_e[(size_t)l * p.E + e2];
                const double L1 = p.mp.Lg[(size_t)l * p.G + g1], L2 = p.mp.Lg[(size_t)l * p.G + g2];
                const double dl = w2 - w1;                                    // moved onto g1
                dload = (float)(2.0 * dl * (L1 - L2) + 2.0 * dl * dl);        // the mean cancels
                dcomm = (fabsf(t12.y) - fabsf(t11.y)) + (fabsf(t21.y) - fabsf(t22.y));
                const float* mt = p.t.m + (size_t)l * p.E * GP;
                const float m11 = p.has_M ? mt[i11] : p.M_scalar, m12 = p.has_M ? mt[i12] : p.M_scalar;
                const float m21 = p.has_M ? mt[i21] : p.M_scalar, m22 = p.has_M ? mt[i22] : p.M_scalar;
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
    if (p.best) {
        unsigned long long key = nan ? ~0ull : ((unsigned long long)ordered_u32(dJ + 0.0f) << 32) | (unsigned long long)(uint32_t)(i & 0xffffffffll);
        const unsigned act = __activemask();
        const int l0 = __shfl_sync(act, l, __ffs(act) - 1);
        if (act == 0xffffffffu && __all_sync(act, l == l0)) {      // one atomic per warp instead of 32 on one address
            for (int o = 16; o > 0; o >>= 1) {
                const unsigned long long other = __shfl_xor_sync(0xffffffffu, key, o);
                key = other < key ? other : key;
            }
            if ((threadIdx.x & 31) == 0 && key != ~0ull) atomicMin(p.best + l, key);
        } else if (key != ~0ull) {
            atomicMin(p.best + l, key);
        }
    }
}

// The whole neighbourhood of `cur` in canonical order (l, a < b): one block per (layer, range of
// row pairs).  The layer's per-slot rows -- communication cost of the slot's expert on every rank (sign =
// x0 hosts it there), its load share w, U = L[rank] - w, the ranks hosting it -- are staged in shared
// memory (pitch G+1: lanes walk b, so rows fall in distinct banks); a warp's 32 results are staged too
// and leave as five fully coalesced 128-byte stores.
//   dC_load = 2 (w2 - w1) (U1 - U2)                 (= 2 d (L1 - L2) + 2 d^2 with d = w2 - w1; double)
//   dC_comm = (c[e1,g2] - c[e1,g1]) + (c[e2,g1] - c[e2,g2])
//   dC_mig  = 2 M (n11 + n22 - n12 - n21), n = "x0 hosts the cell" (scalar M; with a table the four M's with those signs)
//   dmaxload from the layer's three largest rank loads, in fp32 (compared relative to the largest load)
// Same rank or same expert: zeros.  A second copy of an expert on a rank: NaN.  No data-dependent branch.
constexpr int kMoveAllThreads = 512;

__host__ __device__ inline size_t move_all_smem_bytes(int NS, int G, int has_M) {
    size_t b = sizeof(float) * (size_t)NS * (G + 1) * (has_M ? 2 : 1);   // Cs (+ Ms)
    b = (b + 15) & ~size_t(15);
    b += (sizeof(double) * 2 + sizeof(unsigned long long) + sizeof(uint32_t)) * (size_t)NS;   // w, U, cmask, (e | g << 16)
    b = (b + 15) & ~size_t(15);
    b += sizeof(float) * 64;                                                        // rank loads (fp32)
    b += sizeof(float) * (kMoveAllThreads / 32) * 160;                              // output staging
    b += sizeof(unsigned long long) * (kMoveAllThreads / 32);                       // block argmin
    return b;
}

struct MoveSlotsParams {
    int L, E, G, sp, lgG, has_M;
    const int16_t* cur;
    PlaceTables t;
    MovePrep mp;
};

// one thread per (slot, rank) cell of a layer: the layer's tables re-indexed by slot
__global__ void __launch_bounds__(256) move_slots_kernel(const MoveSlotsParams p) {
    const int NS = p.G * p.sp, GP = place_gp(p.G);
    const int l = blockIdx.y, i = blockIdx.x * 256 + threadIdx.x;
    if (i >= NS * p.G) return;
    const int j = i >> p.lgG, g = i & (p.G - 1);
    int e = p.cur[(size_t)l * NS + j];
    if (e < 0 || e >= p.E) e = 0;                                      // flagged by move_prep_kernel
    const size_t src = (size_t)l * p.E * GP + tab_idx(p.E, e, g), dst = ((size_t)l * NS + j) * p.G + g;
    p.mp.slotC[dst] = p.t.wc[src].y;
    if (p.has_M) p.mp.slotM[dst] = p.t.m[src];
    if (g == 0) {
        const double w = p.t.w_e[(size_t)l * p.E + e];
        p.mp.slot_w[(size_t)l * NS + j] = w;
        p.mp.slot_u[(size_t)l * NS + j] = p.mp.Lg[(size_t)l * p.G + j / p.sp] - w;
        p.mp.slot_cm[(size_t)l * NS + j] = p.mp.cmask[(size_t)l * p.E + e];
        p.mp.slot_eg[(size_t)l * NS + j] = make_int2(e, j / p.sp);
    }
}

struct MoveAllParams {
    int L, E, G, sp, has_M;
    int lgG;                            // log2(G)
    int tasks_per_block;                // warp tasks (a row pair) per block
    float alpha, beta, gamma, M_scalar;
    const int16_t* cur;
    PlaceTables t;
    MovePrep mp;
    float* delta;                       // [L * NS*(NS-1)/2, 5]
    unsigned long long* best;           // [L] | nullptr
};

// Work split: row a of the pair triangle (all b > a) has NS-1-a moves, so a warp task is the row
// pair {a, NS-2-a} -- NS-1 moves whatever a is.  Inside a row the lanes walk b: everything that
// depends on a (expert, rank, load, its table row) is warp-uniform, and the results of 32
// consecutive b are contiguous in `delta`.
template <bool kHasM>
__global__ void __launch_bounds__(kMoveAllThreads, 2048 / kMoveAllThreads / 2) move_all_kernel(const MoveAllParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int NS = p.G * p.sp, PITCH = p.G + 1;
    const int l = blockIdx.y, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    float* Cs = reinterpret_cast<float*>(smem_raw);
    float* Ms = Cs + (size_t)NS * PITCH;
    size_t off = sizeof(float) * (size_t)NS * PITCH * (kHasM ? 2 : 1);
    off = (off + 15) & ~size_t(15);
    double* ws = reinterpret_cast<double*>(smem_raw + off); off += sizeof(double) * NS;
    double* us = reinterpret_cast<double*>(smem_raw + off); off += sizeof(double) * NS;
    unsigned long long* cms = reinterpret_cast<unsigned long long*>(smem_raw + off); off += sizeof(unsigned long long) * NS;
    uint32_t* eg = reinterpret_cast<uint32_t*>(smem_raw + off); off += sizeof(uint32_t) * NS;
    off = (off + 15) & ~size_t(15);
    float* Lf = reinterpret_cast<float*>(smem_raw + off); off += sizeof(float) * 64;
    float* stage = reinterpret_cast<float*>(smem_raw + off) + warp * 160; off += sizeof(float) * (kMoveAllThreads / 32) * 160;
    unsigned long long* bests = reinterpret_cast<unsigned long long*>(smem_raw + off);

    const int npairs = NS * (NS - 1) / 2;
    const bool poisoned = (*p.mp.bad != 0) || (*p.t.bad != 0);
    for (int j = tid; j < NS; j += kMoveAllThreads) {
        const int2 s = p.mp.slot_eg[(size_t)l * NS + j];
        eg[j] = (uint32_t)s.x | ((uint32_t)s.y << 16);
        ws[j] = p.mp.slot_w[(size_t)l * NS + j];
        us[j] = p.mp.slot_u[(size_t)l * NS + j];
        cms[j] = p.mp.slot_cm[(size_t)l * NS + j];
    }
    if (tid < p.G) Lf[tid] = (float)p.mp.Lg[(size_t)l * p.G + tid];
    {   // coalesced 16-byte reads of the [NS][G] rows, written at pitch G+1
        const float4* src = reinterpret_cast<const float4*>(p.mp.slotC + (size_t)l * NS * p.G);
        const float4* srcm = reinterpret_cast<const float4*>(p.mp.slotM + (size_t)l * NS * p.G);
        for (int i = tid; i < NS * p.G / 4; i += kMoveAllThreads) {
            const int j = (i * 4) >> p.lgG, g = (i * 4) & (p.G - 1);
            const float4 v = src[i];
            float* d = Cs + j * PITCH + g;
            d[0] = v.x; d[1] = v.y; d[2] = v.z; d[3] = v.w;
            if constexpr (kHasM) {
                const float4 m = srcm[i];
                float* dm = Ms + j * PITCH + g;
                dm[0] = m.x; dm[1] = m.y; dm[2] = m.z; dm[3] = m.w;
            }
        }
    }
    __syncthreads();
    // the three largest rank loads of the layer (fp32) and their ranks
    float top[3]; int top_g[3];
#pragma unroll
    for (int q = 0; q < 3; ++q) { top[q] = (float)p.mp.top[l * 4 + q]; top_g[q] = p.mp.top_g[l * 4 + q]; }
    const float alpha = p.alpha, beta = p.beta, gamma = p.gamma, M2 = 2.0f * p.M_scalar;
    const float ov_nan = poisoned ? CUDART_NAN_F : 0.0f;

    const int n_tasks = NS / 2;                                         // NS-1 rows: (NS-1+1)/2 pairs
    const int t_begin = blockIdx.x * p.tasks_per_block, t_end = min(n_tasks, t_begin + p.tasks_per_block);
    unsigned long long best = ~0ull;
    for (int task = t_begin + warp; task < t_end; task += kMoveAllThreads / 32) {
        for (int half = 0; half < 2; ++half) {
            const int a = half == 0 ? task : NS - 2 - task;
            if (half == 1 && a <= task) break;                          // middle row already done
            const uint32_t s1 = eg[a];
            const int e1 = (int)(s1 & 0xffffu), g1 = (int)(s1 >> 16);
            const double w1 = ws[a], U1 = us[a];
            const unsigned long long cm1 = cms[a];
            const float* Ca = Cs + a * PITCH;
            const float t11 = Ca[g1];
            const uint32_t n11 = __float_as_uint(t11) >> 31;
            const float L1f = Lf[g1], w1f = (float)w1;
            // largest load among the ranks other than g1 (and than g2, decided per lane)
            const float r0v = top_g[0] != g1 ? top[0] : top[1];
            const int r0g = top_g[0] != g1 ? top_g[0] : top_g[1];
            const float r1v = (top_g[0] != g1 && top_g[1] != g1) ? top[1] : top[2];
            const int row0 = a * NS - a * (a + 1) / 2 - a - 1;           // pair index of (a, b) = row0 + b
            for (int bb = a + 1; bb < NS; bb += 32) {
                const int b = min(bb + lane, NS - 1);                    // lanes past the row repeat its last move (not stored)
                const uint32_t s2 = eg[b];
                const int e2 = (int)(s2 & 0xffffu), g2 = (int)(s2 >> 16);
                const bool same = (g1 == g2) || (e1 == e2);
                const bool dup = (((cm1 >> g2) | (cms[b] >> g1)) & 1ull) != 0;
                const float* Cb = Cs + b * PITCH;
                const float t12 = Ca[g2], t21 = Cb[g1], t22 = Cb[g2];
                const double w2 = ws[b];
                const double dl = w2 - w1;                                // load moved onto g1
                float dload = (float)((dl + dl) * (U1 - us[b]));          // 2 d (L1 - L2) + 2 d^2: the mean cancels
                float dcomm = (fabsf(t12) - fabsf(t11)) + (fabsf(t21) - fabsf(t22));
                float dmig;
                if constexpr (kHasM) {
                    const float* Ma = Ms + a * PITCH; const float* Mb = Ms + b * PITCH;
                    // leaving a cell x0 has: +M, leaving a cell x0 lacks: -M; entering: the opposite
                    const float m11 = __uint_as_float(__float_as_uint(Ma[g1]) ^ (~__float_as_uint(t11) & 0x80000000u));
                    const float m12 = __uint_as_float(__float_as_uint(Ma[g2]) ^ (__float_as_uint(t12) & 0x80000000u));
                    const float m22 = __uint_as_float(__float_as_uint(Mb[g2]) ^ (~__float_as_uint(t22) & 0x80000000u));
                    const float m21 = __uint_as_float(__float_as_uint(Mb[g1]) ^ (__float_as_uint(t21) & 0x80000000u));
                    dmig = (m11 + m12) + (m22 + m21);
                } else {
                    const int k = (int)(n11 + (__float_as_uint(t22) >> 31)) - (int)((__float_as_uint(t12) >> 31) + (__float_as_uint(t21) >> 31));
                    dmig = M2 * (float)k;
                }
                const float dlf = (float)w2 - w1f;
                const float rest = (g2 == r0g) ? r1v : r0v;
                float dmax = fmaxf(fmaxf(L1f + dlf, Lf[g2] - dlf), rest) - top[0];
                float dJ = __fmaf_rn(gamma, dmig, __fmaf_rn(beta, dload, alpha * dcomm));
                // overrides: zeros for a move inside one rank / between two copies of one expert, NaN for a second copy on a rank
                const bool use_ov = same || dup || poisoned;
                const float ov = (dup && !same) ? CUDART_NAN_F : ov_nan;
                dJ = use_ov ? ov : dJ; dload = use_ov ? ov : dload; dcomm = use_ov ? ov : dcomm; dmig = use_ov ? ov : dmig; dmax = use_ov ? ov : dmax;
                if (p.best) {
                    const bool cnt = (bb + lane < NS) && !(dJ != dJ);
                    const unsigned long long key = ((unsigned long long)ordered_u32(dJ + 0.0f) << 32) | (unsigned long long)(uint32_t)(l * npairs + row0 + b);
                    best = (cnt && key < best) ? key : best;
                }
                // stage the warp's 32 x 5 results, then write them as contiguous words
                stage[lane * 5 + 0] = dJ; stage[lane * 5 + 1] = dload; stage[lane * 5 + 2] = dcomm; stage[lane * 5 + 3] = dmig; stage[lane * 5 + 4] = dmax;
                __syncwarp();
                const int n_out = min(32, NS - bb) * 5;
                float* out = p.delta + ((size_t)l * npairs + row0 + bb) * 5;
#pragma unroll
                for (int q = 0; q < 5; ++q)
                    if (q * 32 + lane < n_out) __stcs(out + q * 32 + lane, stage[q * 32 + lane]);
                __syncwarp();
            }
        }
    }
    if (p.best) {
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long other = __shfl_xor_sync(0xffffffffu, best, o);
            best = other < best ? other : best;
        }
        if (lane == 0) bests[warp] = best;
        __syncthreads();
        if (tid == 0) {
            for (int w = 1; w < kMoveAllThreads / 32; ++w) best = bests[w] < best ? bests[w] : best;
            if (best != ~0ull) atomicMin(p.best + l, best);
        }
    }
}

// refinement step (gimbal_refine_placement): one thread per layer applies that layer's best exchange when its dJ is
// below minus the rounding margin; the move index is decoded back to the slot pair (a < b, a outer)
__global__ void apply_best_moves_kernel(int L, int NS, float alpha, float beta, float gamma, const int32_t* best, const float* delta,
                                        int16_t* cur, int32_t* applied) {
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= L) return;
    const int bi = best[l];
    if (bi < 0) return;
    const float* d = delta + (size_t)bi * 5;
    const float thr = 1e-4f * (alpha * fabsf(d[2]) + beta * fabsf(d[1]) + gamma * fabsf(d[3]));
    if (!(d[0] < -thr)) return;
    const int npairs = NS * (NS - 1) / 2;
    int r = bi - l * npairs, a = 0;
    while (r >= NS - 1 - a) { r -= NS - 1 - a; ++a; }
    const int b = a + 1 + r;
    int16_t* row = cur + (size_t)l * NS;
    const int16_t t = row[a]; row[a] = row[b]; row[b] = t;
    if (applied) applied[l] += 1;
}

}  // namespace gimbal
