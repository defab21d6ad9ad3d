// a1: router GEMM  logits[i,t,e] = sum_h hidden[i,t,h] * W[layer0+i,e,h]  (+ src_logit_bias),
// bf16 operands, fp32 accumulation in TMEM (BASELINE.json north_star (2)).
//
// Persistent, warp-specialised tcgen05 kernel over all (layer, 128-token tile) pairs of a step:
//   warp 0      TMA producer: hidden tile [128 x 64] + W tile [N/kCG x 64] per k-block into a
//               kStages-deep shared-memory ring (128-byte swizzle), mbarrier full/empty
//   warp 1      MMA issuer (pair leader only): one elected lane issues tcgen05.mma
//               (M = 128*kCG, N = E, K = 16) x 4 per k-block, commits to the ring's empty
//               barriers and, per tile, to the TMEM-full barrier
//   warp 2      TMEM allocator (2 accumulator stages of N fp32 columns)
//   warps 4..7  epilogue: tcgen05.ld 32 lanes x 32 columns -> registers (thread = token row)
//               -> + bias -> logits to HBM and/or fused gating + histogram (a2, a3), then
//               release the accumulator stage
// kCG == 2 pairs two SMs (cta_group::2): each CTA loads its own 128 hidden rows and HALF of
// the W tile, so W traffic out of L2 halves; the leader issues one M=256 MMA for both.
#pragma once
#include "gating.cuh"
#include "stats_update.cuh"
#include "ptx.cuh"

namespace gimbal { constexpr size_t kGemmSmemLimit = 227 * 1024; }

namespace gimbal {

struct GemmParams {
    int n_layers, layer0, T, H, S;
    int m_tiles;                    // ceil(T / (128*kCG))
    int stages;                     // depth of the shared-memory ring (host: gemm_pick_stages)
    int hist_agg;                   // count a warp's tokens by columns when they share one source
    const float* src_logit_bias;    // [L,S,E] | nullptr
    const int32_t* src_offsets;     // [S+1]
    float* logits;                  // [n_layers,T,E] | nullptr
    // fused gating (do_gate != 0)
    int do_gate;
    const float* select_bias;       // [L,E] | nullptr
    int32_t* topk_ids;
    float* topk_w;
    int32_t* A_step;                // [L,S,E]
    unsigned int* zero_word;        // | nullptr: a workspace word this launch clears (stats_update_kernel's block counter)
    int pdl;                        // 0: plain launch; 1: programmatic launch, wait for the predecessor before the first global read;
                                    // 2: (caller's promise that the inputs were ready earlier) wait only before the counts are stored
    int fuse_update;                // store_hist and the call covers all L layers: the pair that stored a layer's counts also runs its
                                    // window / EMA update (`upd`), the last pair finishes the step -- no stats_update_kernel launch
    UpdateParams upd;
    int store_hist;                 // every layer of this call is ONE tile owned by one CTA (pair): the layer's counts are stored
                                    // (the pair's two histograms are added through distributed shared memory), A_step needs no zeroing
    GateParams gp;
    ExpertMap map;
};

constexpr int kGemmThreads = 256;
constexpr int kBlockM = 128;
constexpr int kBlockK = 64;         // 64 bf16 = 128 B = one swizzle row

template <int N, int kCG>
constexpr int gemm_stage_bytes() { return kBlockM * kBlockK * 2 + (N / kCG) * kBlockK * 2; }

constexpr int kGemmAuxBytes = 1024;  // barriers + tmem pointer (<= 12 stages)
constexpr int kGemmMaxStages = 12;

// bytes after the ring: [aux][select_bias N f32][src_offsets S+1 (padded)][hist S*N i32][selection list, when
// ids / weights are written: kListWords x 128 epilogue threads]
// ... [exchange buffers of the epilogue parts, ep > 1: 4 quadrants x [ep][8][32] words]
// words of the histogram region: [S][N] counts (a multiple of 16 words).  The scratch of a fused layer update (UpdateScratch)
// does not live here: it reuses the drained operand ring, which holds at least two stages
__host__ __device__ constexpr size_t gemm_hist_words(int S, int N) { return (size_t)S * N; }
template <int N>
constexpr size_t gemm_tail_bytes(int S, bool out, int ep = 1) {
    return kGemmAuxBytes + sizeof(float) * N + sizeof(int32_t) * (size_t)((S + 1 + 3) & ~3) + sizeof(int32_t) * gemm_hist_words(S, N) +
           (out ? sizeof(int32_t) * (size_t)kListWords * 128 : 0) + (ep > 1 ? sizeof(int32_t) * 4 * (size_t)ep * 8 * 32 : 0);
}
template <int N, int kCG>
inline int gemm_pick_stages(int S, bool out, int ep = 1) {
    const long avail = (long)kGemmSmemLimit - 1024 - (long)gemm_tail_bytes<N>(S, out, ep);
    long s = avail / gemm_stage_bytes<N, kCG>();
    if (s > kGemmMaxStages) s = kGemmMaxStages;
    return (int)s;
}
template <int N, int kCG>
inline size_t gemm_smem_bytes(int S, int stages, bool out, int ep = 1) {
    return 1024 + (size_t)stages * gemm_stage_bytes<N, kCG>() + gemm_tail_bytes<N>(S, out, ep);
}

template <int N>
struct TmemRowSrc {
    uint32_t taddr;                 // lane base | column base of this accumulator stage (+ the first chunk of this epilogue part)
    const float* bias;              // src_logit_bias row for this token (global), from this part's first expert | nullptr
    static constexpr int CH = N < 32 ? N : 32;
    __device__ __forceinline__ void load_raw(int c, uint32_t (&r)[CH]) {
        if constexpr (CH == 32) ptx::tmem_ld_32x32b_x32(taddr + c * 32, r);
        else ptx::tmem_ld_32x32b_x16(taddr + c * 16, r);
        ptx::tmem_ld_wait();
    }
    __device__ __forceinline__ void load(int c, float (&v)[CH]) {
        uint32_t r[CH];
        load_raw(c, r);
#pragma unroll
        for (int i = 0; i < CH; ++i) v[i] = __uint_as_float(r[i]);
        if (bias) {
#pragma unroll
            for (int i = 0; i < CH; i += 4) {
                const float4 b = __ldg(reinterpret_cast<const float4*>(bias + c * CH + i));
                v[i] = __fadd_rn(v[i], b.x); v[i + 1] = __fadd_rn(v[i + 1], b.y);
                v[i + 2] = __fadd_rn(v[i + 2], b.z); v[i + 3] = __fadd_rn(v[i + 3], b.w);
            }
        }
    }
    // order keys overwrite the accumulator columns of this row (the MMA issuer only gets the
    // stage back after the row is done)
    __device__ __forceinline__ void store_keys(int c, const int32_t (&o)[CH]) {
        uint32_t r[CH];
#pragma unroll
        for (int i = 0; i < CH; ++i) r[i] = (uint32_t)o[i];
        if constexpr (CH == 32) ptx::tmem_st_32x32b_x32(taddr + c * 32, r);
        else ptx::tmem_st_32x32b_x16(taddr + c * 16, r);
        ptx::tmem_st_wait();
    }
    __device__ __forceinline__ void load_keys(int c, int32_t (&o)[CH]) {
        uint32_t r[CH];
        load_raw(c, r);
#pragma unroll
        for (int i = 0; i < CH; ++i) o[i] = (int32_t)r[i];
    }
};

template <int N, int kCG, bool kSig, int kEP = 1>
__global__ void __launch_bounds__(128 + 128 * kEP, 1)
router_gemm_kernel(const __grid_constant__ CUtensorMap tmap_a, const __grid_constant__ CUtensorMap tmap_b, const GemmParams p) {
    const int kStages = p.stages;
    constexpr int kABytes = kBlockM * kBlockK * 2;
    constexpr int kBBytes = (N / kCG) * kBlockK * 2;
    constexpr int kStageBytes = kABytes + kBBytes;
    constexpr int kAccCols = N < 32 ? 32 : N;           // TMEM columns per accumulator stage
    constexpr int kTmemCols = 2 * kAccCols < 32 ? 32 : 2 * kAccCols;
    constexpr uint32_t kIdesc = ptx::make_idesc_bf16_f32(128 * kCG, N);
    static_assert(kTmemCols <= 512, "TMEM");

    extern __shared__ unsigned char smem_raw[];
    const uint32_t raw_addr = ptx::smem_u32(smem_raw);
    const uint32_t base = (raw_addr + 1023u) & ~1023u;
    unsigned char* base_ptr = smem_raw + (base - raw_addr);
    // barriers
    const uint32_t aux = base + kStages * kStageBytes;
    const uint32_t full_bar = aux;                       // kStages x 8
    const uint32_t empty_bar = aux + 8 * kStages;        // kStages x 8
    const uint32_t tfull_bar = aux + 16 * kStages;       // 2 x 8
    const uint32_t tempty_bar = tfull_bar + 16;          // 2 x 8
    const uint32_t tmem_slot = tempty_bar + 16;
    uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(base_ptr + kStages * kStageBytes + 16 * kStages + 32);
    float* sb_s = reinterpret_cast<float*>(base_ptr + kStages * kStageBytes + kGemmAuxBytes);
    int32_t* off_s = reinterpret_cast<int32_t*>(sb_s + N);
    int32_t* hist = off_s + ((p.S + 1 + 3) & ~3);
    int32_t* list_s = hist + gemm_hist_words(p.S, N);    // [kListWords][128] (only when ids / weights are written)
    int32_t* xbuf_s = list_s;                            // kEP > 1 (counts only, no list): [4 quadrants][kEP][8][32] exchange words
    constexpr int kThreads = 128 + 128 * kEP, kEpiThreads = 128 * kEP;
    static_assert(kEP == 1 || (N / 32) % kEP == 0, "epilogue parts split the 32-expert chunks of a row");

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t cta_rank = (kCG == 2) ? ptx::cluster_ctarank() : 0u;
    const bool leader = cta_rank == 0;
    const int pair = blockIdx.x / kCG, n_pairs = gridDim.x / kCG;
    const int n_tiles = p.n_layers * p.m_tiles;
    const int num_kb = (p.H + kBlockK - 1) / kBlockK;

    // Launched with programmatic stream serialization in the one-tile-per-layer regime (p.pdl != 0).  pdl == 2: everything up to
    // the store of the counts may overlap the previous kernel of the stream (stats_update_kernel of the step before, which still
    // reads A_step and its block counter); the next kernel may be scheduled right away (it waits for this grid itself).
    if (p.pdl == 2) ptx::griddep_launch_dependents();
    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tmap_a);
        ptx::prefetch_tmap(&tmap_b);
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < kStages; ++s) {
            ptx::mbar_init(full_bar + 8 * s, 1);
            ptx::mbar_init(empty_bar + 8 * s, 1);
        }
        for (int a = 0; a < 2; ++a) {
            ptx::mbar_init(tfull_bar + 8 * a, 1);
            ptx::mbar_init(tempty_bar + 8 * a, 4 * kEP * kCG);   // one arrive per epilogue warp per CTA
        }
        ptx::fence_barrier_init();
    }
    if (warp == 2) {
        ptx::tmem_alloc<kCG>(tmem_slot, kTmemCols);
        ptx::tmem_relinquish<kCG>();
    }
    if (p.pdl == 1) {
        // barriers, TMEM and descriptors are set up: from here on global memory is read, so the predecessor must be complete
        ptx::griddep_wait();
        ptx::griddep_launch_dependents();
    }
    for (int i = threadIdx.x; i <= p.S; i += kThreads) off_s[i] = p.src_offsets[i];
    ptx::tc_fence_before();
    if constexpr (kCG == 2) ptx::cluster_sync(); else __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        // ================= TMA producer =================
        if (lane == 0) {
            const uint64_t pol_a = ptx::policy_evict_first();   // hidden is read exactly once
            const uint64_t pol_b = ptx::policy_evict_last();    // W[l] is re-read by every tile of the layer
            const uint32_t full_leader = (kCG == 2) ? ptx::mapa(full_bar, 0) : full_bar;
            int stage = 0; uint32_t phase = 0;
            for (int tile = pair; tile < n_tiles; tile += n_pairs) {
                const int li = tile / p.m_tiles, mt = tile % p.m_tiles;
                const int m0 = (mt * kCG + (int)cta_rank) * kBlockM;
                const int n0 = (int)cta_rank * (N / kCG);
                for (int kb = 0; kb < num_kb; ++kb) {
                    ptx::mbar_wait(empty_bar + 8 * stage, phase ^ 1);
                    if (leader) ptx::mbar_arrive_expect_tx(full_bar + 8 * stage, kCG * kStageBytes);
                    const uint32_t sa = base + stage * kStageBytes;
                    const uint32_t fb = (kCG == 2) ? full_leader + 8 * stage : full_bar + 8 * stage;
                    ptx::tma_load_3d<kCG>(sa, &tmap_a, fb, kb * kBlockK, m0, li, pol_a);
                    ptx::tma_load_3d<kCG>(sa + kABytes, &tmap_b, fb, kb * kBlockK, n0, p.layer0 + li, pol_b);
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ================= MMA issuer (leader CTA of the pair) =================
        if (leader) {
            int stage = 0; uint32_t phase = 0;
            int it = 0;
            for (int tile = pair; tile < n_tiles; tile += n_pairs, ++it) {
                const int as = it & 1;
                const uint32_t aphase = (it >> 1) & 1;
                if (kCG == 2) ptx::mbar_wait_cluster(tempty_bar + 8 * as, aphase ^ 1);
                else ptx::mbar_wait(tempty_bar + 8 * as, aphase ^ 1);
                ptx::tc_fence_after();
                const uint32_t d_tmem = tmem_base + as * kAccCols;
                for (int kb = 0; kb < num_kb; ++kb) {
                    ptx::mbar_wait(full_bar + 8 * stage, phase);
                    ptx::tc_fence_after();
                    if (lane == 0) {
                        const uint32_t sa = base + stage * kStageBytes;
                        const uint64_t da = ptx::make_sw128_kmajor_desc(sa);
                        const uint64_t db = ptx::make_sw128_kmajor_desc(sa + kABytes);
#pragma unroll
                        for (int k = 0; k < kBlockK / 16; ++k) {
                            // +32 B per K=16 step inside the 128-byte swizzle row (>>4 = 2)
                            ptx::umma_bf16<kCG>(d_tmem, da + 2 * k, db + 2 * k, kIdesc, (kb | k) != 0);
                        }
                        ptx::umma_commit<kCG>(empty_bar + 8 * stage);          // frees the smem slot (both CTAs)
                        if (kb == num_kb - 1) ptx::umma_commit<kCG>(tfull_bar + 8 * as);   // accumulator ready
                    }
                    __syncwarp();
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp >= 4) {
        // ================= epilogue: TMEM -> registers -> logits / gating =================
        const int q = (warp - 4) & 3;                 // TMEM lane quadrant (== warp % 4)
        const int part = (warp - 4) >> 2;             // kEP > 1: which share of the experts (columns) of the rows of quadrant q
        const int ep_tid = threadIdx.x - 128;
        const CrossParts xp{xbuf_s + q * (kEP * 8 * 32), 2 + q, 32 * kEP};
        const uint32_t tempty_leader = (kCG == 2) ? ptx::mapa(tempty_bar, 0) : tempty_bar;
        int it = 0;
        int cur_layer = -1;
        for (int tile = pair; tile < n_tiles; tile += n_pairs, ++it) {
            const int as = it & 1;
            const uint32_t aphase = (it >> 1) & 1;
            const int li = tile / p.m_tiles, mt = tile % p.m_tiles;
            const int layer = p.layer0 + li;
            const int m0 = (mt * kCG + (int)cta_rank) * kBlockM;
            const int t = m0 + q * 32 + lane;
            if (p.do_gate && layer != cur_layer) {
                // new layer: flush the histogram of the previous one, load this layer's select bias
                asm volatile("bar.sync 1, %0;" ::"n"(kEpiThreads) : "memory");
                if (cur_layer >= 0) {
                    int32_t* dst = p.A_step + (size_t)cur_layer * p.S * N;
                    for (int i = ep_tid; i < p.S * N; i += kEpiThreads) {
                        const int32_t c = hist[i];
                        if (c) atomicAdd(dst + i, c);
                    }
                }
                for (int i = ep_tid; i < p.S * N; i += kEpiThreads) hist[i] = 0;
                for (int i = ep_tid; i < N; i += kEpiThreads) sb_s[i] = p.select_bias ? p.select_bias[(size_t)layer * N + i] : 0.0f;
                cur_layer = layer;
                asm volatile("bar.sync 1, %0;" ::"n"(kEpiThreads) : "memory");
            }
            ptx::mbar_wait(tfull_bar + 8 * as, aphase);
            ptx::tc_fence_after();
            const uint32_t taddr = tmem_base + as * kAccCols + ((uint32_t)(q * 32) << 16);
            const int s = find_source(off_s, p.S, min(t, p.T - 1));
            const float* bias = p.src_logit_bias ? p.src_logit_bias + ((size_t)layer * p.S + s) * N : nullptr;
            TmemRowSrc<N> src{taddr, bias};
            if constexpr (kEP > 1) {
                // counts only (the host picks kEP > 1 when neither logits nor ids / weights are asked for): this warp gates the
                // experts [part * N / kEP, (part + 1) * N / kEP) of its quadrant's rows and meets the other parts in shared memory
                constexpr int kPartCols = N / kEP;
                TmemRowSrc<N> psrc{taddr + part * kPartCols, bias ? bias + part * kPartCols : nullptr};
                int32_t ids[kTopK];
                float w[kTopK];
                const bool uni = p.hist_agg && __all_sync(0xffffffffu, s == __shfl_sync(0xffffffffu, s, 0));
                gate_row<N, kSig, false, TmemRowSrc<N>, kEP, true>(p.gp, sb_s, psrc, t < p.T, hist + s * N, nullptr, 0, ids, w, part, uni, &xp);
            } else {
            if (p.logits) {
                constexpr int CH = TmemRowSrc<N>::CH;
                float v[CH];
                float* orow = p.logits + ((size_t)li * p.T + t) * N;
#pragma unroll
                for (int c = 0; c < N / CH; ++c) {
                    src.load(c, v);
                    if (t < p.T) {
#pragma unroll
                        for (int i = 0; i < CH; i += 4)
                            *reinterpret_cast<float4*>(orow + c * CH + i) = make_float4(v[i], v[i + 1], v[i + 2], v[i + 3]);
                    }
                }
            }
            if (p.do_gate) {
                int32_t ids[kTopK];
                float w[kTopK];
                const bool valid = t < p.T;
                if (p.topk_ids || p.topk_w || p.map.rep_off) {
                    gate_row<N, kSig, true>(p.gp, sb_s, src, valid, hist + s * N, list_s + ep_tid, 128, ids, w);
                    if (valid && p.topk_ids) {
                        int32_t* o = p.topk_ids + ((size_t)li * p.T + t) * p.gp.k;
#pragma unroll
                        for (int j = 0; j < kTopK; ++j)
                            if (j < p.gp.k) o[j] = ids[j];
                    }
                    if (valid && p.topk_w) {
                        float* o = p.topk_w + ((size_t)li * p.T + t) * p.gp.k;
#pragma unroll
                        for (int j = 0; j < kTopK; ++j)
                            if (j < p.gp.k) o[j] = w[j];
                    }
                    if (valid && p.map.rep_off) map_row<N>(p.map, layer, li, p.T, t, p.gp.k, ids);
                } else {
                    // rows past T follow the last row's source; a warp whose 32 rows share one source counts by columns
                    const bool uni = p.hist_agg && __all_sync(0xffffffffu, s == __shfl_sync(0xffffffffu, s, 0));
                    gate_row<N, kSig, false>(p.gp, sb_s, src, valid, hist + s * N, nullptr, 0, ids, w, 0, uni);
                }
            }
            }
            // release this accumulator stage to the MMA issuer
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) {
                if (kCG == 2) ptx::mbar_arrive_cluster(tempty_leader + 8 * as);
                else ptx::mbar_arrive(tempty_bar + 8 * as);
            }
        }
        if (p.do_gate && cur_layer >= 0 && !p.store_hist) {
            asm volatile("bar.sync 1, %0;" ::"n"(kEpiThreads) : "memory");
            int32_t* dst = p.A_step + (size_t)cur_layer * p.S * N;
            for (int i = ep_tid; i < p.S * N; i += kEpiThreads) {
                const int32_t c = hist[i];
                if (c) atomicAdd(dst + i, c);
            }
        }
    }

    // ================= teardown =================
    ptx::tc_fence_before();
    if constexpr (kCG == 2) ptx::cluster_sync(); else __syncthreads();
    if (blockIdx.x == 0 && threadIdx.x == 32 && p.zero_word) {
        ptx::griddep_wait();
        *p.zero_word = 0u;                                                       // consumed by the next kernel of the stream
    }
    if (p.do_gate && p.store_hist) {
        if (warp >= 4 && leader) ptx::griddep_wait();                            // the previous step's stats_update_kernel is done with A_step
        // one tile per layer, one CTA (pair) per tile: the barrier above made both histograms of the pair complete and visible;
        // the leader adds its peer's through distributed shared memory and STORES the layer's counts (zeros included)
        int64_t step_now = 0;
        if (warp >= 4 && leader) {
            const int ep_tid = threadIdx.x - 128;
            const int layer = p.layer0 + pair;                                   // tile == pair, m_tiles == 1
            if (p.fuse_update) step_now = *p.upd.step_counter;                   // (behind the wait above; its latency hides in the loop below)
            int32_t* dst = p.A_step + (size_t)layer * p.S * N;
            const uint32_t peer = (kCG == 2) ? ptx::mapa(ptx::smem_u32(hist), 1) : 0u;
            const int n4 = p.S * N / 4;                                          // N % 4 == 0, hist is 16-byte aligned
#pragma unroll 4
            for (int i = ep_tid; i < n4; i += kEpiThreads) {
                int4 c = reinterpret_cast<const int4*>(hist)[i];
                if constexpr (kCG == 2) {
                    const uint4 o = ptx::ld_shared_cluster_v4(peer + 16u * (uint32_t)i);
                    c.x += (int32_t)o.x; c.y += (int32_t)o.y; c.z += (int32_t)o.z; c.w += (int32_t)o.w;
                }
                reinterpret_cast<int4*>(dst)[i] = c;
                reinterpret_cast<int4*>(hist)[i] = c;                            // the layer's counts stay here for the update below
            }
        }
        if constexpr (kCG == 2) ptx::cluster_sync();                             // the peer's shared memory stays until it was read
        if (p.fuse_update && warp >= 4 && leader) {
            // a4 + a5 of this layer right here, from the counts in `hist`; scratch = the (drained) operand ring
            asm volatile("bar.sync 1, %0;" ::"n"(kEpiThreads) : "memory");
            static_assert(2 * gemm_stage_bytes<N, kCG>() >= (int)sizeof(UpdateScratch), "the scratch of the fused update must fit two ring stages");
            UpdateScratch& sh = *reinterpret_cast<UpdateScratch*>(base_ptr);
            const int32_t* hc = hist;
            stats_update_layer(p.upd, p.layer0 + pair, (int)threadIdx.x - 128, kEpiThreads, sh, step_now,
                               [] { asm volatile("bar.sync 1, %0;" ::"n"(kEpiThreads) : "memory"); },
                               [hc](int s, int e) { return hc[s * N + e]; });
        }
    }
    if (warp == 2) ptx::tmem_dealloc<kCG>(tmem_base, kTmemCols);
}

}  // namespace gimbal
