// a6 with the expert -> rank candidate encoding (`EXPERT_TO_RANK_U8`, [P,L,E] uint8, one byte per
// expert = the rank that hosts it; only for placements without replicas, NS == E).  Half the candidate bytes of the
// slot -> expert int16 encoding; the price is that a rank's load becomes a scatter-add (PAPER.md:236 sums over the
// experts of a rank, and here the experts of a rank are not contiguous).
//
// Lane <-> EPL consecutive experts (EPL = E/32, at least 4), so B[e] and x0's rank of e sit in registers, and the layer's
// table is staged rank-major and expert-swizzled, ct[g][k * LPC + li] for expert e = EPL * li + k, so that the lookup
// of (e, rank(e)) by the lanes of a candidate falls in distinct banks.  Rank loads are accumulated with shared-memory
// atomics on a per-warp [G] array; the capacity check (every rank hosts exactly slots_per_rank experts) counts beside it.
#pragma once
#include "placement.cuh"

namespace gimbal {

struct E2RParams {
    int P, L, G, sp, chunk, check;
    float M_scalar;
    const uint8_t* cand;                // [P,L,E]
    const float* M;                     // caller's [L,E,G] | nullptr
    PlaceTables t;
    float4* partial;
};

constexpr int kE2RWarps = 8;

inline size_t e2r_smem_bytes(int E, int G, bool has_M) {
    return sizeof(float) * (size_t)G * E * (has_M ? 2 : 1) + (size_t)kE2RWarps * 8 * 64 * 8;
}

template <int E, bool kHasM>
__global__ void __launch_bounds__(kE2RWarps * 32) place_score_e2r_kernel(const E2RParams p) {
    constexpr int EPL = E >= 128 ? E / 32 : 4;          // experts per lane
    constexpr int LPC = E / EPL;                        // lanes per candidate
    constexpr int UPW = 32 / LPC;                       // candidates per warp
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int G = p.G, l = blockIdx.y;
    float* ct_s = reinterpret_cast<float*>(smem_raw);                                     // [G][E] c, sign = x0 hosts e on g
    float* mt_s = ct_s + (size_t)G * E;                                                   // [G][E] (kHasM) cost of e being on g
    float* acc_s = ct_s + (size_t)G * E * (kHasM ? 2 : 1);                                // [warps][UPW][64] loads, then counts
    int* cnt_all = reinterpret_cast<int*>(acc_s + kE2RWarps * UPW * 64);
    const size_t tab = (size_t)l * (place_gp(G) / 32) * E * 32;
    for (int idx = threadIdx.x; idx < G * E; idx += kE2RWarps * 32) {
        const int g = idx / E, pos = idx % E, k = pos / LPC, li = pos % LPC, e = EPL * li + k;
        const float c = p.t.wc[tab + tab_idx(E, e, g)].y;
        ct_s[idx] = c;
        if constexpr (kHasM) {
            // r = 1: expert e either stays on x0's rank (nothing) or leaves it and enters g: M[e,g0] + M[e,g]
            const int g0e = __ffsll((long long)p.t.pmask[(size_t)l * E + e]) - 1;
            const float* Ml = p.M + ((size_t)l * E + e) * G;
            mt_s[idx] = (__float_as_int(c) < 0 || g0e < 0) ? 0.0f : __fadd_rn(Ml[g], Ml[g0e]);
        }
    }
    for (int i = threadIdx.x; i < kE2RWarps * UPW * 64; i += kE2RWarps * 32) { acc_s[i] = 0.0f; cnt_all[i] = 0; }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, sub = lane / LPC, li = lane % LPC;
    float bw[EPL];
#pragma unroll
    for (int k = 0; k < EPL; ++k) bw[k] = p.t.wc[tab + tab_idx(E, EPL * li + k, 0)].x;    // B[e] (r = 1)
    __syncthreads();
    float* lg = acc_s + (warp * UPW + sub) * 64;
    int* cnt = cnt_all + (warp * UPW + sub) * 64;
    const double Gd = (double)G, sumB = p.t.sumB[l];
    const int p_begin = blockIdx.x * p.chunk, p_end = min(p.P, p_begin + p.chunk);
    for (int pc = p_begin + warp * UPW; pc < p_end; pc += kE2RWarps * UPW) {
        const int c = pc + sub;
        const bool active = c < p_end;
        float comm = 0.0f, mig = 0.0f;
        int kept = 0;
        bool bad = false;
        if (active) {
            const uint8_t* row = p.cand + ((size_t)c * p.L + l) * E + EPL * li;
            uint32_t wv[EPL / 4];
            if constexpr (EPL == 8) { const uint2 v = __ldcs(reinterpret_cast<const uint2*>(row)); wv[0] = v.x; wv[1] = v.y; }
            else wv[0] = __ldcs(reinterpret_cast<const uint32_t*>(row));
#pragma unroll
            for (int k = 0; k < EPL; ++k) {
                uint32_t g = (wv[k >> 2] >> (8 * (k & 3))) & 0xffu;
                bad |= g >= (uint32_t)G;
                g = min(g, (uint32_t)G - 1u);
                const int at = (int)g * E + k * LPC + li;
                const float v = ct_s[at];
                comm += fabsf(v);
                kept += (int)(__float_as_uint(v) >> 31);
                if constexpr (kHasM) mig += mt_s[at];
                atomicAdd(lg + g, bw[k]);
                if (p.check) atomicAdd(cnt + g, 1);
            }
        }
        __syncwarp();
        float sq = 0.0f, mx = 0.0f;
        for (int g = li; g < G; g += LPC) {
            const float v = lg[g];
            const float d = (float)((double)v * Gd - sumB);
            sq = __fmaf_rn(d, d, sq);
            mx = fmaxf(mx, v);
            if (p.check && cnt[g] != p.sp) bad = true;            // a rank over (hence another under) capacity
            lg[g] = 0.0f; cnt[g] = 0;
        }
        __syncwarp();
#pragma unroll
        for (int o = LPC >> 1; o > 0; o >>= 1) {
            sq += __shfl_xor_sync(0xffffffffu, sq, o);
            comm += __shfl_xor_sync(0xffffffffu, comm, o);
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
            kept += __shfl_xor_sync(0xffffffffu, kept, o);
            bad |= __shfl_xor_sync(0xffffffffu, (int)bad, o) != 0;
            if constexpr (kHasM) mig += __shfl_xor_sync(0xffffffffu, mig, o);
        }
        if constexpr (!kHasM) mig = p.M_scalar * (float)(2 * (E - kept));
        if (active && li == 0)
            p.partial[(size_t)c * p.L + l] = bad ? make_float4(CUDART_NAN_F, CUDART_NAN_F, CUDART_NAN_F, CUDART_NAN_F) : make_float4(sq, comm, mig, mx);
    }
}

}  // namespace gimbal
