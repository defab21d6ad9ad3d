// C-ABI entry points of libgimbal (include/gimbal.h): argument validation, workspace
// carving, TMA descriptor encoding and kernel launches.  Every step of the hot path runs in
// the kernels of this directory; there is no CPU fallback.
#include <cuda.h>
#include <cuda_runtime.h>
#include <cuda_bf16.h>

#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

#define GIMBAL_DEFINE_STATS_UPDATE_KERNEL
#include "host_common.h"
#include "greedy.cuh"
#include "placement.cuh"
#include "placement_e2r.cuh"
#include "sched.cuh"
#include "stats_update.cuh"

using namespace gimbal;

namespace gimbal {
int ktime_enable(int on);
int ktime_elapsed(int which, float* ms);
int64_t launches();
void copy_last_error(char* buf, size_t n);
}

namespace {

constexpr int kHostCtxSlots = 64;

// ---- workspace carving ---------------------------------------------------------------------
struct Carver {
    unsigned char* base;
    size_t off = 0;
    explicit Carver(void* p) : base(static_cast<unsigned char*>(p)) {}
    template <class T>
    T* take(size_t n) {
        off = (off + 255) & ~size_t(255);
        T* r = base ? reinterpret_cast<T*>(base + off) : nullptr;
        off += n * sizeof(T);
        return r;
    }
};

int launch_gemm(const RouteArgs& a) {
    switch (a.cfg->E) {
        case 16: return launch_gemm_e16(a);
        case 32: return launch_gemm_e32(a);
        case 64: return launch_gemm_e64(a);
        case 128: return launch_gemm_e128(a);
        case 256: return launch_gemm_e256(a);
    }
    return fail(GIMBAL_ERR_UNSUPPORTED, "E=%d not in {16,32,64,128,256}", a.cfg->E);
}

int launch_gate(const RouteArgs& a) {
    switch (a.cfg->E) {
        case 16: return launch_gate_e16(a);
        case 32: return launch_gate_e32(a);
        case 64: return launch_gate_e64(a);
        case 128: return launch_gate_e128(a);
        case 256: return launch_gate_e256(a);
    }
    return fail(GIMBAL_ERR_UNSUPPORTED, "E=%d not in {16,32,64,128,256}", a.cfg->E);
}

int validate_router_cfg(const gimbal_router_cfg* c) {
    if (!c) return fail(GIMBAL_ERR_INVALID_ARG, "cfg is NULL");
    if (c->L < 1 || c->H < 1 || c->S < 1 || c->k < 1) return fail(GIMBAL_ERR_INVALID_ARG, "L, H, S, k must be >= 1");
    if (c->E != 16 && c->E != 32 && c->E != 64 && c->E != 128 && c->E != 256)
        return fail(GIMBAL_ERR_UNSUPPORTED, "E=%d not in {16,32,64,128,256}", c->E);
    if (c->k > GIMBAL_MAX_TOPK || c->k > c->E) return fail(GIMBAL_ERR_UNSUPPORTED, "k=%d (max %d, <= E)", c->k, GIMBAL_MAX_TOPK);
    if (c->S > GIMBAL_MAX_SOURCES) return fail(GIMBAL_ERR_UNSUPPORTED, "S=%d (max %d)", c->S, GIMBAL_MAX_SOURCES);
    if (c->H % 64 != 0) return fail(GIMBAL_ERR_UNSUPPORTED, "H=%d must be a multiple of 64", c->H);
    if (c->score_fn != GIMBAL_SCORE_SOFTMAX && c->score_fn != GIMBAL_SCORE_SIGMOID)
        return fail(GIMBAL_ERR_INVALID_ARG, "score_fn=%d", c->score_fn);
    if (c->n_groups < 1) return fail(GIMBAL_ERR_INVALID_ARG, "n_groups=%d", c->n_groups);
    if (c->n_groups > 1) {
        if (c->E % c->n_groups != 0 || c->E / c->n_groups != 32)
            return fail(GIMBAL_ERR_UNSUPPORTED, "group-limited routing needs E/n_groups == 32 (E=%d, n_groups=%d)", c->E, c->n_groups);
        if (c->topk_groups < 1 || c->topk_groups > c->n_groups) return fail(GIMBAL_ERR_INVALID_ARG, "topk_groups=%d", c->topk_groups);
        if (c->group_score_topn != 1 && c->group_score_topn != 2)
            return fail(GIMBAL_ERR_UNSUPPORTED, "group_score_topn=%d not in {1,2}", c->group_score_topn);
        if (c->topk_groups * 32 < c->k) return fail(GIMBAL_ERR_INVALID_ARG, "topk_groups*32 < k");
    }
    return GIMBAL_OK;
}

struct RouteWs {
    double* partial;           // [L,S]
    unsigned int* done;        // [1] (+pad)
};

size_t route_ws_carve(const gimbal_router_cfg* c, void* ws, RouteWs* out) {
    Carver cv(ws);
    RouteWs w;
    w.partial = cv.take<double>((size_t)c->L * c->S);
    w.done = cv.take<unsigned int>(64);
    if (out) *out = w;
    return cv.off + 256;
}

// process-wide switches set through gimbal_set_option (tests and A/B measurements); defaults = production
std::atomic<int> g_opt[GIMBAL_OPT_COUNT_] = {{0}, {1}, {0}, {0}, {1}, {1}, {0}, {1}, {1}};

int pick_cta_group(int T) {
    const int forced = g_opt[GIMBAL_OPT_CTA_GROUP].load(std::memory_order_relaxed);
    if (forced == 1 || forced == 2) return forced;
    return T > 128 ? 2 : 1;
}

int pick_fuse() { return g_opt[GIMBAL_OPT_FUSE_GATE].load(std::memory_order_relaxed); }

// ------------------------------------------------------------------------------------------
static int validate_place_cfg(const gimbal_placement_cfg* c) {
    if (!c) return fail(GIMBAL_ERR_INVALID_ARG, "cfg is NULL");
    if (c->L < 1 || c->E < 1 || c->G < 1 || c->slots_per_rank < 1 || c->S < 1) return fail(GIMBAL_ERR_INVALID_ARG, "L, E, G, slots_per_rank, S must be >= 1");
    if (c->E > kMaxE) return fail(GIMBAL_ERR_UNSUPPORTED, "E=%d (max %d)", c->E, kMaxE);
    if (c->G > kMaxG || (c->G & (c->G - 1))) return fail(GIMBAL_ERR_UNSUPPORTED, "G=%d must be a power of two <= %d", c->G, kMaxG);
    if (c->slots_per_rank > 16) return fail(GIMBAL_ERR_UNSUPPORTED, "slots_per_rank=%d (max 16)", c->slots_per_rank);
    if (c->S > GIMBAL_MAX_SOURCES) return fail(GIMBAL_ERR_UNSUPPORTED, "S=%d (max %d)", c->S, GIMBAL_MAX_SOURCES);
    if ((long)c->G * c->slots_per_rank < c->E) return fail(GIMBAL_ERR_INVALID_ARG, "G*slots_per_rank < E");
    if (c->counts_dtype != GIMBAL_COUNTS_I32 && c->counts_dtype != GIMBAL_COUNTS_F32) return fail(GIMBAL_ERR_INVALID_ARG, "counts_dtype=%d", c->counts_dtype);
    if (c->E % 2 != 0) return fail(GIMBAL_ERR_UNSUPPORTED, "E must be even");
    // candidate / placement rows [NS] int16 are read as 32-bit words: an odd row length would misalign every other row
    if (((long)c->G * c->slots_per_rank) % 2 != 0) return fail(GIMBAL_ERR_UNSUPPORTED, "G*slots_per_rank=%ld must be even", (long)c->G * c->slots_per_rank);
    if (c->encoding != GIMBAL_ENC_SLOT_TO_EXPERT_I16 && c->encoding != GIMBAL_ENC_EXPERT_TO_RANK_U8) return fail(GIMBAL_ERR_INVALID_ARG, "encoding=%d", c->encoding);
    if (c->flags & ~GIMBAL_PLACE_TRUSTED) return fail(GIMBAL_ERR_INVALID_ARG, "flags=0x%x has bits this library does not know", c->flags);
    return GIMBAL_OK;
}

struct PlaceWs {
    PlaceTables t;
    float4* partial;                // [P,L]
    uint8_t* status;                // [P,L] place_check_kernel's verdicts
    unsigned long long* best;       // [max(L,1)]
    MovePrep mp;
};

static size_t place_ws_carve(const gimbal_placement_cfg* c, int P, void* ws, PlaceWs* out) {
    Carver cv(ws);
    PlaceWs w{};
    const int GP = place_gp(c->G);
    const size_t LE = (size_t)c->L * c->E;
    const size_t NSl = (size_t)c->L * c->G * c->slots_per_rank;
    w.t.wc = cv.take<float2>(LE * GP);
    w.t.c_s = cv.take<float>(LE * GP);
    w.t.w_f = cv.take<float>(LE);
    w.t.m = cv.take<float>(LE * GP);
    w.t.mu = cv.take<uint32_t>(LE * GP);
    w.t.mx0 = cv.take<float>(NSl);
    w.t.c_raw = cv.take<float>(LE * c->G);
    w.t.b_raw = cv.take<double>(LE);
    w.t.w_e = cv.take<double>(LE);
    w.t.sumB = cv.take<double>(c->L);
    w.t.r = cv.take<int32_t>(LE);
    w.t.pmask = cv.take<uint64_t>(LE);
    w.t.bad = cv.take<int32_t>(64);
    w.partial = cv.take<float4>((size_t)P * c->L);
    w.status = cv.take<uint8_t>((size_t)P * c->L);
    w.best = cv.take<unsigned long long>(c->L + 1);
    w.mp.Lg = cv.take<double>((size_t)c->L * c->G);
    w.mp.top = cv.take<double>((size_t)c->L * 4);
    w.mp.top_g = cv.take<int32_t>((size_t)c->L * 4);
    w.mp.cmask = cv.take<uint64_t>(LE);
    w.mp.bad = cv.take<int32_t>(64);
    w.mp.slotC = cv.take<float>(NSl * c->G);
    w.mp.slotM = cv.take<float>(NSl * c->G);
    w.mp.slot_w = cv.take<double>(NSl);
    w.mp.slot_u = cv.take<double>(NSl);
    w.mp.slot_cm = cv.take<uint64_t>(NSl);
    w.mp.slot_eg = cv.take<int2>(NSl);
    if (out) *out = w;
    return cv.off + 256;
}

static int launch_tables(const gimbal_placement_cfg* c, const void* A, const void* B, const float* D, const float* M, float M_scalar,
                         const int16_t* prev, const PlaceWs& w, cudaStream_t stream) {
    CUDA_TRY(cudaMemsetAsync(w.t.bad, 0, sizeof(int32_t), stream));
    TableParams tp{};
    tp.L = c->L; tp.E = c->E; tp.G = c->G; tp.sp = c->slots_per_rank; tp.S = c->S; tp.counts_f32 = c->counts_dtype == GIMBAL_COUNTS_F32;
    tp.A = A; tp.B = B; tp.D = D; tp.M = M; tp.M_scalar = M_scalar; tp.prev = prev; tp.t = w.t;
    const size_t smem_a = sizeof(float) * (size_t)c->S * c->E;           // the layer's [S][E] counts, at most 64 KB
    if (smem_a > 24 * 1024) CUDA_TRY(cudaFuncSetAttribute(place_tables_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_a));
    place_tables_kernel<<<dim3(c->L, kTableSplit), 256, smem_a, stream>>>(tp);
    LAUNCH_CHECK("place_tables_kernel");
    return GIMBAL_OK;
}

template <bool kHasM>
static int launch_score_generic(const ScoreParams& sp, dim3 grid, size_t smem, cudaStream_t stream) {
    auto kern = place_score_generic_kernel<kHasM>;
    CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ktime_begin(GIMBAL_KERNEL_SCORE, stream);
    kern<<<grid, kScoreThreads, smem, stream>>>(sp);
    ktime_end(GIMBAL_KERNEL_SCORE, stream);
    LAUNCH_CHECK("place_score_generic_kernel");
    return GIMBAL_OK;
}

template <int SP, int G, int E, bool kHasM, bool kCheck>
static int launch_score_v(const ScoreParams& sp, dim3 grid, size_t smem, cudaStream_t stream) {
    auto kern = place_score_kernel<SP, G, E, kHasM, kCheck>;
    CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ktime_begin(GIMBAL_KERNEL_SCORE, stream);
    kern<<<grid, kScoreThreads, smem, stream>>>(sp);
    ktime_end(GIMBAL_KERNEL_SCORE, stream);
    LAUNCH_CHECK("place_score_kernel");
    return GIMBAL_OK;
}

// the 9 x 32 x 256 shape, scalar M, scoring only: candidate rows by TMA (place_score_tma_kernel)
static int launch_score_tma(const ScoreParams& sp, dim3 grid, cudaStream_t stream) {
    CUtensorMap tm;
    int rc = make_tmap_rows_i16_4d(&tm, sp.cand, 72, 4, (uint64_t)sp.L, (uint64_t)sp.P, 80, kScoreU);
    if (rc) return rc;
    const size_t smem = place_score_tma_smem_bytes();
    CUDA_TRY(cudaFuncSetAttribute(place_score_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ktime_begin(GIMBAL_KERNEL_SCORE, stream);
    place_score_tma_kernel<<<grid, kScoreThreads, smem, stream>>>(sp, tm);
    ktime_end(GIMBAL_KERNEL_SCORE, stream);
    LAUNCH_CHECK("place_score_tma_kernel");
    return GIMBAL_OK;
}

template <int SP, int G, int E>
static int launch_score(const ScoreParams& sp, bool check, dim3 grid, size_t smem, cudaStream_t stream) {
    if (check) return sp.has_M ? launch_score_v<SP, G, E, true, true>(sp, grid, smem, stream) : launch_score_v<SP, G, E, false, true>(sp, grid, smem, stream);
    return sp.has_M ? launch_score_v<SP, G, E, true, false>(sp, grid, smem, stream) : launch_score_v<SP, G, E, false, false>(sp, grid, smem, stream);
}

template <int E>
static int launch_e2r_e(const E2RParams& ep, bool has_M, dim3 grid, size_t smem, cudaStream_t stream) {
    auto kern = has_M ? place_score_e2r_kernel<E, true> : place_score_e2r_kernel<E, false>;
    CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ktime_begin(GIMBAL_KERNEL_SCORE, stream);
    kern<<<grid, kE2RWarps * 32, smem, stream>>>(ep);
    ktime_end(GIMBAL_KERNEL_SCORE, stream);
    LAUNCH_CHECK("place_score_e2r_kernel");
    return GIMBAL_OK;
}

static int launch_e2r(const gimbal_placement_cfg* c, int P, const uint8_t* cand, const float* M, float M_scalar, const PlaceTables& t,
                      float4* partial, size_t smem, int sms, cudaStream_t stream) {
    E2RParams ep{};
    ep.P = P; ep.L = c->L; ep.G = c->G; ep.sp = c->slots_per_rank; ep.check = !(c->flags & GIMBAL_PLACE_TRUSTED);
    ep.M_scalar = M_scalar; ep.cand = cand; ep.M = M; ep.t = t; ep.partial = partial;
    const int per_sm = (int)((kSmemLimit - 1024) / (smem + 1024)) < 1 ? 1 : (int)((kSmemLimit - 1024) / (smem + 1024));
    int nchunk = (per_sm > 4 ? 4 : per_sm) * sms / c->L;
    const int maxc = (P + kE2RWarps - 1) / kE2RWarps;
    if (nchunk > maxc) nchunk = maxc;
    if (nchunk < 1) nchunk = 1;
    ep.chunk = (P + nchunk - 1) / nchunk;
    dim3 grid((P + ep.chunk - 1) / ep.chunk, c->L);
    switch (c->E) {
        case 16: return launch_e2r_e<16>(ep, M != nullptr, grid, smem, stream);
        case 32: return launch_e2r_e<32>(ep, M != nullptr, grid, smem, stream);
        case 64: return launch_e2r_e<64>(ep, M != nullptr, grid, smem, stream);
        case 128: return launch_e2r_e<128>(ep, M != nullptr, grid, smem, stream);
        case 256: return launch_e2r_e<256>(ep, M != nullptr, grid, smem, stream);
    }
    return fail(GIMBAL_ERR_UNSUPPORTED, "EXPERT_TO_RANK_U8 needs E in {16,32,64,128,256}, got %d", c->E);
}

// inverse of a slot -> expert placement: one block per layer, thread e collects expert e's slots in
// ascending order (deterministic)
__global__ void __launch_bounds__(256) expert_map_kernel(int E, int NS, const int16_t* placement, int32_t* rep_off, int16_t* rep_slots,
                                                         int32_t* status) {
    __shared__ int cnt_s[kMaxE + 1];
    __shared__ int16_t pl_s[kMaxG * 16];
    const int l = blockIdx.x, tid = threadIdx.x;
    for (int e = tid; e <= E; e += 256) cnt_s[e] = 0;
    __syncthreads();
    bool bad = false;
    for (int j = tid; j < NS; j += 256) {
        const int e = placement[(size_t)l * NS + j];
        pl_s[j] = (int16_t)e;
        if (e < 0 || e >= E) bad = true; else atomicAdd(&cnt_s[e + 1], 1);
    }
    if (bad && status) atomicOr(status, 1);
    __syncthreads();
    if (tid == 0)
        for (int e = 0; e < E; ++e) cnt_s[e + 1] += cnt_s[e];          // exclusive offsets in cnt_s[0..E]
    __syncthreads();
    for (int e = tid; e <= E; e += 256) rep_off[(size_t)l * (E + 1) + e] = cnt_s[e];
    for (int e = tid; e < E; e += 256) {
        int pos = cnt_s[e];
        for (int j = 0; j < NS; ++j)
            if (pl_s[j] == e) rep_slots[(size_t)l * NS + pos++] = (int16_t)j;
    }
}

}  // namespace

extern "C" {

int gimbal_version(void) { return GIMBAL_ABI_VERSION; }

void gimbal_last_error(char* buf, size_t n) {
    if (!buf || n == 0) return;
    gimbal::copy_last_error(buf, n);
}

int64_t gimbal_launch_count(void) { return gimbal::launches(); }

int gimbal_set_option(int option, int value) {
    if (option < 0 || option >= GIMBAL_OPT_COUNT_) return fail(GIMBAL_ERR_INVALID_ARG, "option %d", option);
    const bool three = option == GIMBAL_OPT_CTA_GROUP || option == GIMBAL_OPT_EPI_PARTS || option == GIMBAL_OPT_PDL;
    if (three && (value < 0 || value > 2)) return fail(GIMBAL_ERR_INVALID_ARG, "option %d takes 0, 1 or 2", option);
    if (!three && value != 0 && value != 1) return fail(GIMBAL_ERR_INVALID_ARG, "option %d takes 0 or 1", option);
    g_opt[option].store(value, std::memory_order_relaxed);
    return GIMBAL_OK;
}

int gimbal_get_option(int option, int* value) {
    if (option < 0 || option >= GIMBAL_OPT_COUNT_ || !value) return fail(GIMBAL_ERR_INVALID_ARG, "option %d", option);
    *value = g_opt[option].load(std::memory_order_relaxed);
    return GIMBAL_OK;
}

int gimbal_kernel_timing(int enable) { return gimbal::ktime_enable(enable); }

int gimbal_kernel_elapsed_ms(int which, float* ms) { return gimbal::ktime_elapsed(which, ms); }

size_t gimbal_route_stats_workspace_bytes(const gimbal_router_cfg* cfg, int n_layers, int T) {
    (void)n_layers; (void)T;
    if (!cfg) return 0;
    return route_ws_carve(cfg, nullptr, nullptr);
}

size_t gimbal_route_stats_result_bytes(const gimbal_router_cfg* cfg) {
    if (!cfg) return 0;
    return sizeof(int32_t) * (size_t)cfg->L * cfg->S * cfg->E + 4 * (size_t)cfg->L * cfg->E + 2 * sizeof(float) * (size_t)cfg->S;
}

int gimbal_route_stats(const gimbal_router_cfg* cfg, int layer0, int n_layers, int T, const void* hidden, const void* w_router,
                       const float* select_bias, const float* src_logit_bias, const int32_t* src_offsets, int logits_mode,
                       float* logits, int32_t* topk_ids, float* topk_w, const int16_t* cur_placement, const int32_t* dp_of_rank,
                       int G, int slots_per_rank, gimbal_stats_state* st, const gimbal_expert_map* map, void* workspace,
                       size_t workspace_bytes, gimbal_stream_t stream_) {
    int rc = validate_router_cfg(cfg);
    if (rc) return rc;
    if (map && (!map->rep_off || !map->rep_slots || !map->phys_ids || map->NS < cfg->E))
        return fail(GIMBAL_ERR_INVALID_ARG, "expert map needs rep_off, rep_slots, phys_ids and NS >= E");
    if (layer0 < 0 || n_layers < 1 || layer0 + n_layers > cfg->L) return fail(GIMBAL_ERR_INVALID_ARG, "layer range [%d,%d) outside [0,%d)", layer0, layer0 + n_layers, cfg->L);
    if (T < 0) return fail(GIMBAL_ERR_INVALID_ARG, "T=%d", T);
    if (!src_offsets) return fail(GIMBAL_ERR_INVALID_ARG, "src_offsets is NULL");
    if (!st) return fail(GIMBAL_ERR_INVALID_ARG, "state is NULL");
    // a state laid out by another header (round 1: step_counter [1], this field `reserved` = 0) would be written out of bounds
    if (st->abi_version != GIMBAL_ABI_VERSION)
        return fail(GIMBAL_ERR_INVALID_ARG, "state->abi_version=%d, this library is %d: rebuild against include/gimbal.h (step_counter is i64[2])",
                    st->abi_version, GIMBAL_ABI_VERSION);
    if (!st->A_step || !st->step_counter || !st->B) return fail(GIMBAL_ERR_INVALID_ARG, "state: A_step / B / step_counter is NULL");
    if (st->mode == GIMBAL_MODE_WINDOW) {
        if (!st->A_win || !st->A_pub || !st->B_pub || st->window_len < 1) return fail(GIMBAL_ERR_INVALID_ARG, "WINDOW mode needs A_win, A_pub, B_pub, window_len >= 1");
    } else if (st->mode == GIMBAL_MODE_EMA) {
        if (!st->A_ema) return fail(GIMBAL_ERR_INVALID_ARG, "EMA mode needs A_ema");
    } else return fail(GIMBAL_ERR_INVALID_ARG, "state mode=%d", st->mode);
    if (logits_mode != GIMBAL_LOGITS_NONE && logits_mode != GIMBAL_LOGITS_OUT && logits_mode != GIMBAL_LOGITS_IN)
        return fail(GIMBAL_ERR_INVALID_ARG, "logits_mode=%d", logits_mode);
    if (logits_mode != GIMBAL_LOGITS_NONE && !logits) return fail(GIMBAL_ERR_INVALID_ARG, "logits is NULL");
    if (logits_mode != GIMBAL_LOGITS_NONE && (reinterpret_cast<uintptr_t>(logits) & 15)) return fail(GIMBAL_ERR_INVALID_ARG, "logits must be 16-byte aligned");
    if (logits_mode != GIMBAL_LOGITS_IN) {
        if (!hidden || !w_router) return fail(GIMBAL_ERR_INVALID_ARG, "hidden / w_router is NULL");
        if ((reinterpret_cast<uintptr_t>(hidden) & 15) || (reinterpret_cast<uintptr_t>(w_router) & 15))
            return fail(GIMBAL_ERR_INVALID_ARG, "hidden / w_router must be 16-byte aligned");
        // the fused epilogue reads a token's bias row with 16-byte loads
        if (src_logit_bias && (reinterpret_cast<uintptr_t>(src_logit_bias) & 15)) return fail(GIMBAL_ERR_INVALID_ARG, "src_logit_bias must be 16-byte aligned");
    }
    if ((cur_placement != nullptr) != (dp_of_rank != nullptr)) return fail(GIMBAL_ERR_INVALID_ARG, "cur_placement and dp_of_rank go together");
    if (cur_placement) {
        if (G < 1 || G > kMaxG || slots_per_rank < 1 || (long)G * slots_per_rank < cfg->E || !st->pressure_raw || !st->pressure_rel)
            return fail(GIMBAL_ERR_INVALID_ARG, "pressure needs 1 <= G <= 64, G*slots >= E, pressure_raw/rel");
    }
    RouteWs ws;
    const size_t need = route_ws_carve(cfg, workspace, &ws);
    if (!workspace || workspace_bytes < need) return fail(GIMBAL_ERR_WORKSPACE, "workspace %zu < %zu bytes", workspace_bytes, need);
    rc = require_device();
    if (rc) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);

    // a3 accumulates into A_step with atomics: zero the slice of this call -- unless every layer is one tile with a CTA (pair)
    // of its own (small-batch regime: T <= 256, n_layers <= pairs), where the fused router kernel stores a layer's counts
    const int cg_pick = pick_cta_group(T);
    const bool hist_stored = T > 0 && logits_mode != GIMBAL_LOGITS_IN && pick_fuse() && (size_t)cfg->S * cfg->E * 4 <= 64 * 1024 && T <= 128 * cg_pick &&
                             n_layers <= device_info().sms / cg_pick;
    if (!hist_stored)
        CUDA_TRY(cudaMemsetAsync(st->A_step + (size_t)layer0 * cfg->S * cfg->E, 0, sizeof(int32_t) * (size_t)n_layers * cfg->S * cfg->E, stream));
    // whole-step call in that regime: the pair that stores a layer's counts also runs the layer's update (a4-a5) and the last pair
    // finishes the step; its layer counter is the second word of state->step_counter (zero between calls), so nothing is zeroed
    // and no stats_update_kernel is launched
    const bool update_fused = hist_stored && layer0 == 0 && n_layers == cfg->L && g_opt[GIMBAL_OPT_FUSE_UPDATE].load(std::memory_order_relaxed);
    UpdateParams u{};
    u.L = cfg->L; u.S = cfg->S; u.E = cfg->E; u.G = G; u.sp = slots_per_rank;
    u.mode = st->mode; u.window_len = st->window_len; u.ema_decay = st->ema_decay;
    u.A_step = st->A_step; u.A_win = st->A_win; u.A_pub = st->A_pub; u.B_pub = st->B_pub; u.A_ema = st->A_ema; u.B = st->B;
    u.pressure_raw = st->pressure_raw; u.pressure_rel = st->pressure_rel; u.step_counter = st->step_counter; u.status = st->status;
    u.cur_placement = cur_placement; u.dp_of_rank = dp_of_rank; u.partial = ws.partial;
    u.done_counter = update_fused ? reinterpret_cast<unsigned int*>(st->step_counter + 1) : ws.done;
    // stats_update_kernel's block counter starts at 0: the router kernel of this call clears it where there is one, else a memset
    const bool gemm_clears = layer0 == 0 && T > 0 && logits_mode != GIMBAL_LOGITS_IN && !update_fused;
    if (layer0 == 0 && !gemm_clears && !update_fused) CUDA_TRY(cudaMemsetAsync(ws.done, 0, sizeof(unsigned int), stream));

    if (T > 0) {
        RouteArgs a{};
        a.cfg = cfg; a.layer0 = layer0; a.n_layers = n_layers; a.T = T; a.hidden = hidden; a.w_router = w_router;
        a.select_bias = select_bias; a.src_logit_bias = src_logit_bias; a.src_offsets = src_offsets;
        a.topk_ids = topk_ids; a.topk_w = topk_w; a.A_step = st->A_step; a.stream = stream;
        a.zero_word = gemm_clears ? ws.done : nullptr;
        a.upd = update_fused ? &u : nullptr;
        if (map) { a.rep_off = map->rep_off; a.rep_slots = map->rep_slots; a.phys_ids = map->phys_ids; a.map_NS = map->NS; }
        a.cta_group = cg_pick;
        a.store_hist = hist_stored;
        a.pdl = g_opt[GIMBAL_OPT_PDL].load(std::memory_order_relaxed);
        a.hist_agg = g_opt[GIMBAL_OPT_HIST_AGG].load(std::memory_order_relaxed);
        {
            // epilogue parts: auto = 2 when no CTA (pair) gets more than two tiles, i.e. when the epilogue cannot hide behind the MMAs
            const int forced = g_opt[GIMBAL_OPT_EPI_PARTS].load(std::memory_order_relaxed);
            const int rows = 128 * a.cta_group;
            const long tiles = (long)n_layers * ((T + rows - 1) / rows);
            const int pairs = device_info().sms / a.cta_group;
            a.epi_parts = forced ? forced : (tiles <= 2L * pairs ? 2 : 1);
        }
        if (logits_mode == GIMBAL_LOGITS_IN) {
            a.logits = logits;
            rc = launch_gate(a);
            if (rc) return rc;
        } else {
            // fused epilogue needs the block histogram next to the ring; fall back to two kernels otherwise
            const bool can_fuse = pick_fuse() && (size_t)cfg->S * cfg->E * 4 <= 64 * 1024;   // every supported (S, E) fits
            if (can_fuse) {
                a.logits = logits_mode == GIMBAL_LOGITS_OUT ? logits : nullptr;
                a.fuse_gate = 1;
                rc = launch_gemm(a);
                if (rc) return rc;
            } else {
                if (logits_mode != GIMBAL_LOGITS_OUT) return fail(GIMBAL_ERR_UNSUPPORTED, "unfused path needs logits_mode OUT (a logits buffer)");
                a.logits = logits; a.fuse_gate = 0;
                rc = launch_gemm(a);
                if (rc) return rc;
                rc = launch_gate(a);
                if (rc) return rc;
            }
        }
    }

    if (layer0 + n_layers == cfg->L && !update_fused) {
        cudaLaunchConfig_t lc{};
        lc.gridDim = dim3(cfg->L); lc.blockDim = dim3(kUpdateThreads); lc.dynamicSmemBytes = 0; lc.stream = stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        lc.attrs = at; lc.numAttrs = g_opt[GIMBAL_OPT_PDL].load(std::memory_order_relaxed) ? 1 : 0;
        CUDA_TRY(cudaLaunchKernelEx(&lc, stats_update_kernel, u));
        LAUNCH_CHECK("stats_update_kernel");
    }
    return GIMBAL_OK;
}

// ---- gimbal_route_stats_static: the scratch of the a4-a5 update lives in the library ------------------
// One array per device that has this module loaded, zero at load, kept until the process exits.  In HOST code the name below is
// only the handle that cudaGetSymbolAddress understands; the pointer a kernel may use is what that call returns, per device.
static __device__ __align__(256) unsigned char gimbal_static_scratch[GIMBAL_STATIC_SCRATCH_BYTES];

namespace {
constexpr int kStaticMaxDevices = 64;
struct StaticScratchDev {
    void* ptr = nullptr;     // device address of gimbal_static_scratch on this device (set-up done when non-null)
    size_t layout = 0;       // bytes the previous call on this device carved (0: none yet)
};
std::mutex g_static_mu;
StaticScratchDev g_static_dev[kStaticMaxDevices];
}  // namespace

int gimbal_route_stats_static(const gimbal_router_cfg* cfg, int layer0, int n_layers, int T, const void* hidden, const void* w_router,
                              const float* select_bias, const float* src_logit_bias, const int32_t* src_offsets, int logits_mode,
                              float* logits, int32_t* topk_ids, float* topk_w, const int16_t* cur_placement, const int32_t* dp_of_rank,
                              int G, int slots_per_rank, gimbal_stats_state* st, const gimbal_expert_map* map, gimbal_stream_t stream_) {
    int rc = validate_router_cfg(cfg);
    if (rc) return rc;
    const size_t need = route_ws_carve(cfg, nullptr, nullptr);
    if (need > sizeof gimbal_static_scratch)
        return fail(GIMBAL_ERR_WORKSPACE,
                    "gimbal_route_stats_static: L=%d x S=%d needs %zu bytes of scratch, the built-in array holds %zu (L*S <= 8128); "
                    "use gimbal_route_stats with a workspace of your own",
                    cfg->L, cfg->S, need, sizeof gimbal_static_scratch);
    rc = require_device();
    if (rc) return rc;
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(GIMBAL_ERR_UNSUPPORTED, "gimbal_route_stats_static: device ordinal %d (max %d)", dev, kStaticMaxDevices - 1);
    void* scratch = nullptr;
    bool relayout = false;
    {
        std::lock_guard<std::mutex> lk(g_static_mu);
        StaticScratchDev& d = g_static_dev[dev];
        if (!d.ptr) {
            // set-up, once per device, with that device current: ask the runtime where the array lives on it
            void* p = nullptr;
            const cudaError_t e = cudaGetSymbolAddress(&p, gimbal_static_scratch);
            if (e != cudaSuccess || !p)
                return fail(GIMBAL_ERR_CUDA, "cudaGetSymbolAddress(gimbal_static_scratch) on device %d: %s", dev, cudaGetErrorString(e));
            d.ptr = p;
        }
        scratch = d.ptr;
        relayout = d.layout != need;
        d.layout = need;
    }
    // the array keeps the previous call's contents: under a new layout the layer counter may sit where partials were
    if (relayout) CUDA_TRY(cudaMemsetAsync(scratch, 0, need, static_cast<cudaStream_t>(stream_)));
    return gimbal_route_stats(cfg, layer0, n_layers, T, hidden, w_router, select_bias, src_logit_bias, src_offsets, logits_mode, logits,
                              topk_ids, topk_w, cur_placement, dp_of_rank, G, slots_per_rank, st, map, scratch,
                              sizeof gimbal_static_scratch, stream_);
}

struct gimbal_host_ctx {
    int device;
    cudaStream_t copy_stream;
    cudaEvent_t ev_start;
    cudaEvent_t ev_copied[kHostCtxSlots], ev_done[kHostCtxSlots];
};

// destroys whatever a (possibly half-built) context holds; handles that were never created are null
static void host_ctx_release(gimbal_host_ctx* c) {
    for (int i = 0; i < kHostCtxSlots; ++i) {
        if (c->ev_copied[i]) cudaEventDestroy(c->ev_copied[i]);
        if (c->ev_done[i]) cudaEventDestroy(c->ev_done[i]);
    }
    if (c->ev_start) cudaEventDestroy(c->ev_start);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    delete c;
}

int gimbal_host_ctx_create(gimbal_host_ctx** out) {
    if (!out) return fail(GIMBAL_ERR_INVALID_ARG, "ctx out pointer is NULL");
    *out = nullptr;
    int rc = require_device();
    if (rc) return rc;
    gimbal_host_ctx* c = new (std::nothrow) gimbal_host_ctx();     // value-initialised: every handle starts null
    if (!c) return fail(GIMBAL_ERR_CUDA, "out of host memory");
    // a failure half-way must not leak the stream and the events made so far
    cudaError_t e = cudaGetDevice(&c->device);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming);
    for (int i = 0; i < kHostCtxSlots && e == cudaSuccess; ++i) {
        e = cudaEventCreateWithFlags(&c->ev_copied[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_done[i], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) {
        host_ctx_release(c);
        return fail(GIMBAL_ERR_CUDA, "gimbal_host_ctx_create: %s", cudaGetErrorString(e));
    }
    *out = c;
    return GIMBAL_OK;
}

int gimbal_host_ctx_destroy(gimbal_host_ctx* c) {
    if (!c) return GIMBAL_OK;
    cudaStreamSynchronize(c->copy_stream);
    host_ctx_release(c);
    return GIMBAL_OK;
}

int gimbal_route_stats_host(gimbal_host_ctx* ctx, const gimbal_router_cfg* cfg, int T, const void* hidden_host,
                            const int32_t* src_offsets_host, void* hidden_stage, size_t hidden_stage_bytes,
                            int32_t* src_offsets_stage, const void* w_router, const float* select_bias, const float* src_logit_bias,
                            const int16_t* cur_placement, const int32_t* dp_of_rank, int G, int slots_per_rank,
                            gimbal_stats_state* st, void* result_host, void* workspace, size_t workspace_bytes,
                            gimbal_stream_t stream_) {
    int rc = validate_router_cfg(cfg);
    if (rc) return rc;
    if (!ctx) return fail(GIMBAL_ERR_INVALID_ARG, "host ctx is NULL (gimbal_host_ctx_create)");
    if (!hidden_host || !src_offsets_host || !hidden_stage || !src_offsets_stage || !result_host || !st)
        return fail(GIMBAL_ERR_INVALID_ARG, "NULL host / staging pointer");
    const size_t layer_bytes = (size_t)T * cfg->H * 2;
    if (T < 1) return fail(GIMBAL_ERR_INVALID_ARG, "T=%d", T);
    const size_t slots = hidden_stage_bytes / layer_bytes;
    if (slots < 2) return fail(GIMBAL_ERR_WORKSPACE, "hidden_stage must hold at least 2 layers (%zu bytes)", 2 * layer_bytes);
    rc = require_device();
    if (rc) return rc;
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev != ctx->device) return fail(GIMBAL_ERR_INVALID_ARG, "host ctx belongs to device %d, current device is %d", ctx->device, dev);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    // the context's second stream carries the copies so that layer i+1 streams in while layer i computes
    cudaStream_t copy_stream = ctx->copy_stream;
    const size_t nslot = slots > (size_t)kHostCtxSlots ? (size_t)kHostCtxSlots : slots;
    CUDA_TRY(cudaMemcpyAsync(src_offsets_stage, src_offsets_host, sizeof(int32_t) * (cfg->S + 1), cudaMemcpyHostToDevice, stream));
    CUDA_TRY(cudaEventRecord(ctx->ev_start, stream));
    CUDA_TRY(cudaStreamWaitEvent(copy_stream, ctx->ev_start, 0));
    for (int l = 0; l < cfg->L; ++l) {
        const size_t slot = (size_t)l % nslot;
        unsigned char* dst = static_cast<unsigned char*>(hidden_stage) + slot * layer_bytes;
        if ((size_t)l >= nslot) CUDA_TRY(cudaStreamWaitEvent(copy_stream, ctx->ev_done[slot], 0));   // slot's previous layer consumed
        CUDA_TRY(cudaMemcpyAsync(dst, static_cast<const unsigned char*>(hidden_host) + (size_t)l * layer_bytes, layer_bytes,
                                 cudaMemcpyHostToDevice, copy_stream));
        CUDA_TRY(cudaEventRecord(ctx->ev_copied[slot], copy_stream));
        CUDA_TRY(cudaStreamWaitEvent(stream, ctx->ev_copied[slot], 0));
        rc = gimbal_route_stats(cfg, l, 1, T, dst, w_router, select_bias, src_logit_bias, src_offsets_stage, GIMBAL_LOGITS_NONE,
                                nullptr, nullptr, nullptr, cur_placement, dp_of_rank, G, slots_per_rank, st, nullptr, workspace,
                                workspace_bytes, stream_);
        if (rc) return rc;
        CUDA_TRY(cudaEventRecord(ctx->ev_done[slot], stream));
    }
    unsigned char* out = static_cast<unsigned char*>(result_host);
    const size_t nA = sizeof(int32_t) * (size_t)cfg->L * cfg->S * cfg->E, nB = 4 * (size_t)cfg->L * cfg->E, nP = sizeof(float) * cfg->S;
    CUDA_TRY(cudaMemcpyAsync(out, st->A_step, nA, cudaMemcpyDeviceToHost, stream));
    CUDA_TRY(cudaMemcpyAsync(out + nA, st->B, nB, cudaMemcpyDeviceToHost, stream));
    if (st->pressure_raw && st->pressure_rel) {
        CUDA_TRY(cudaMemcpyAsync(out + nA + nB, st->pressure_raw, nP, cudaMemcpyDeviceToHost, stream));
        CUDA_TRY(cudaMemcpyAsync(out + nA + nB + nP, st->pressure_rel, nP, cudaMemcpyDeviceToHost, stream));
    }
    CUDA_TRY(cudaStreamSynchronize(stream));
    return GIMBAL_OK;
}

size_t gimbal_eval_placements_workspace_bytes(const gimbal_placement_cfg* cfg, int P) {
    if (!cfg || P < 0) return 0;
    return place_ws_carve(cfg, P, nullptr, nullptr);
}

size_t gimbal_eval_moves_workspace_bytes(const gimbal_placement_cfg* cfg) {
    if (!cfg) return 0;
    return place_ws_carve(cfg, 0, nullptr, nullptr);
}

int gimbal_eval_placements(const gimbal_placement_cfg* cfg, int P, const void* candidates, const void* A, const void* B,
                           const float* D, const float* M, float M_scalar, const int16_t* prev, float* out, int32_t* argmin,
                           void* workspace, size_t workspace_bytes, gimbal_stream_t stream_) {
    int rc = validate_place_cfg(cfg);
    if (rc) return rc;
    if (P < 0) return fail(GIMBAL_ERR_INVALID_ARG, "P=%d", P);
    if (!A || !B || !D || !prev || (P > 0 && (!candidates || !out))) return fail(GIMBAL_ERR_INVALID_ARG, "NULL argument");
    if (reinterpret_cast<uintptr_t>(candidates) & 15) return fail(GIMBAL_ERR_INVALID_ARG, "candidates must be 16-byte aligned");
    const int NS = cfg->G * cfg->slots_per_rank;
    const bool e2r = cfg->encoding == GIMBAL_ENC_EXPERT_TO_RANK_U8;
    if (e2r && NS != cfg->E) return fail(GIMBAL_ERR_INVALID_ARG, "EXPERT_TO_RANK_U8 needs G*slots_per_rank == E (no replicas)");
    if (e2r && cfg->E % 4 != 0) return fail(GIMBAL_ERR_UNSUPPORTED, "EXPERT_TO_RANK_U8 needs E %% 4 == 0");
    PlaceWs w;
    const size_t need = place_ws_carve(cfg, P, workspace, &w);
    if (!workspace || workspace_bytes < need) return fail(GIMBAL_ERR_WORKSPACE, "workspace %zu < %zu bytes", workspace_bytes, need);
    const int GP = place_gp(cfg->G);
    const size_t smem = e2r ? e2r_smem_bytes(cfg->E, cfg->G, M != nullptr) : (size_t)cfg->E * GP * (M ? 12 : 8);
    if (smem > kSmemLimit) return fail(GIMBAL_ERR_UNSUPPORTED, "E=%d G=%d with an M table needs %zu B of shared memory", cfg->E, cfg->G, smem);
    const size_t smem_chk = place_check_smem_bytes(cfg->G);
    rc = require_device();
    if (rc) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    if (argmin) {
        fill_u64_kernel<<<1, 32, 0, stream>>>(w.best, ~0ull, 1);
        LAUNCH_CHECK("fill_u64_kernel");
    }
    if (P > 0) {
        rc = launch_tables(cfg, A, B, D, M, M_scalar, prev, w, stream);
        if (rc) return rc;
        const int sms = device_info().sms;
        if (e2r) {
            rc = launch_e2r(cfg, P, static_cast<const uint8_t*>(candidates), M, M_scalar, w.t, w.partial, smem, sms, stream);
            if (rc) return rc;
        } else {
            ScoreParams sp{};
            sp.P = P; sp.L = cfg->L; sp.E = cfg->E; sp.G = cfg->G; sp.sp = cfg->slots_per_rank; sp.M_scalar = M_scalar; sp.has_M = M != nullptr;
            sp.cand = static_cast<const int16_t*>(candidates); sp.t = w.t; sp.partial = w.partial; sp.status = w.status;
            sp.force_general = g_opt[GIMBAL_OPT_CHECK_SCORES_ALL].load(std::memory_order_relaxed);
            const bool trusted = (cfg->flags & GIMBAL_PLACE_TRUSTED) != 0;
            // the five configuration shapes (slots per rank, ranks, experts) have specialised kernels, which also validate
            // in the same pass (kCheck); any other shape: the shape-generic scoring kernel, then place_check_kernel
            const long key = g_opt[GIMBAL_OPT_SCORE_GENERIC].load(std::memory_order_relaxed)
                                 ? 0 : (long)cfg->slots_per_rank * 1000000 + cfg->G * 1000 + cfg->E;
            const bool fast = key == 9032256 || key == 8016128 || key == 8008064 || key == 4064256 || key == 4004016;
            const bool fused = fast && !trusted && smem + place_score_mask_bytes(cfg->G, cfg->E) <= kSmemLimit;   // else: separate check kernel
            const size_t smem_k = smem + (fused ? place_score_mask_bytes(cfg->G, cfg->E) : 0);
            // one wave: two resident blocks per SM (one when a block needs more than half the shared memory)
            const int per_sm = (fast && 2 * smem_k + 2048 <= kSmemLimit) ? 2 : 1;
            int nchunk = per_sm * sms / cfg->L;
            const int units_per_pass = (kScoreThreads / 32) * (cfg->G < 32 ? 32 / cfg->G : 1);
            int max_chunks = (P + units_per_pass - 1) / units_per_pass;
            if (nchunk > max_chunks) nchunk = max_chunks;
            if (nchunk < 1) nchunk = 1;
            sp.chunk = (P + nchunk - 1) / nchunk;
            dim3 grid((P + sp.chunk - 1) / sp.chunk, cfg->L);
            switch (fast ? key : 0) {
                case 9032256:
                    if (!fused && !sp.has_M && g_opt[GIMBAL_OPT_SCORE_TMA].load(std::memory_order_relaxed)) rc = launch_score_tma(sp, grid, stream);
                    else rc = launch_score<9, 32, 256>(sp, fused, grid, smem_k, stream);
                    break;
                case 8016128: rc = launch_score<8, 16, 128>(sp, fused, grid, smem_k, stream); break;
                case 8008064: rc = launch_score<8, 8, 64>(sp, fused, grid, smem_k, stream); break;
                case 4064256: rc = launch_score<4, 64, 256>(sp, fused, grid, smem_k, stream); break;
                case 4004016: rc = launch_score<4, 4, 16>(sp, fused, grid, smem_k, stream); break;
                default: rc = sp.has_M ? launch_score_generic<true>(sp, grid, smem, stream) : launch_score_generic<false>(sp, grid, smem, stream); break;
            }
            if (rc) return rc;
            if (!trusted) {
                CheckParams cp{};
                cp.P = P; cp.L = cfg->L; cp.E = cfg->E; cp.G = cfg->G; cp.sp = cfg->slots_per_rank;
                cp.force_general = sp.force_general;
                cp.M_scalar = M_scalar; cp.cand = sp.cand; cp.prev = prev; cp.M = M; cp.t = w.t; cp.partial = w.partial; cp.status = w.status;
                int nck = 8 * sms / cfg->L;
                const int maxck = (P + kCheckWarps - 1) / kCheckWarps;
                if (nck > maxck) nck = maxck;
                if (nck < 1) nck = 1;
                cp.chunk = (P + nck - 1) / nck;
                const dim3 cgrid((P + cp.chunk - 1) / cp.chunk, cfg->L);
                if (!fused) {
                    // exact validation; overwrites the partials of invalid candidates (NaN) and marks the valid ones whose
                    // replica counts differ from x0's
                    ktime_begin(GIMBAL_KERNEL_CHECK, stream);
                    const int ckey = cfg->slots_per_rank * 10 + (cfg->G > 32 ? 2 : 1);
                    switch (ckey) {
                        case 41: place_check_kernel<4, 1><<<cgrid, kCheckWarps * 32, smem_chk, stream>>>(cp); break;
                        case 42: place_check_kernel<4, 2><<<cgrid, kCheckWarps * 32, smem_chk, stream>>>(cp); break;
                        case 81: place_check_kernel<8, 1><<<cgrid, kCheckWarps * 32, smem_chk, stream>>>(cp); break;
                        case 91: place_check_kernel<9, 1><<<cgrid, kCheckWarps * 32, smem_chk, stream>>>(cp); break;
                        default:
                            if (cfg->G > 32) place_check_kernel<0, 2><<<cgrid, kCheckWarps * 32, smem_chk, stream>>>(cp);
                            else place_check_kernel<0, 1><<<cgrid, kCheckWarps * 32, smem_chk, stream>>>(cp);
                            break;
                    }
                    ktime_end(GIMBAL_KERNEL_CHECK, stream);
                    LAUNCH_CHECK("place_check_kernel");
                }
                // candidates with their own replica counts: scored with the candidate's r
                place_own_r_kernel<<<cgrid, kCheckWarps * 32, smem_chk, stream>>>(cp);
                LAUNCH_CHECK("place_own_r_kernel");
            }
        }
        FinalizeParams fp{};
        fp.P = P; fp.L = cfg->L; fp.G = cfg->G; fp.alpha = cfg->alpha; fp.beta = cfg->beta; fp.gamma = cfg->gamma;
        fp.partial = w.partial; fp.bad_prev = w.t.bad; fp.out = out; fp.best = argmin ? w.best : nullptr;
        place_finalize_kernel<<<(P + 7) / 8, 256, 0, stream>>>(fp);
        LAUNCH_CHECK("place_finalize_kernel");
    }
    if (argmin) {
        best_to_index_kernel<<<1, 32, 0, stream>>>(w.best, argmin, 1);
        LAUNCH_CHECK("best_to_index_kernel");
    }
    return GIMBAL_OK;
}

int gimbal_eval_placements_host(const gimbal_placement_cfg* cfg, int P, const void* candidates_host, void* cand_stage,
                                float* out_stage, const void* A, const void* B, const float* D, const float* M, float M_scalar,
                                const int16_t* prev, float* out_host, int32_t* argmin_host, void* workspace, size_t workspace_bytes,
                                gimbal_stream_t stream_) {
    int rc = validate_place_cfg(cfg);
    if (rc) return rc;
    if (P < 0) return fail(GIMBAL_ERR_INVALID_ARG, "P=%d", P);
    if (!candidates_host || !cand_stage || !out_stage || !out_host) return fail(GIMBAL_ERR_INVALID_ARG, "NULL host / staging pointer");
    PlaceWs w;
    const size_t need = place_ws_carve(cfg, P, workspace, &w);
    if (!workspace || workspace_bytes < need) return fail(GIMBAL_ERR_WORKSPACE, "workspace %zu < %zu bytes", workspace_bytes, need);
    rc = require_device();
    if (rc) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const size_t row = cfg->encoding == GIMBAL_ENC_EXPERT_TO_RANK_U8 ? (size_t)cfg->E : sizeof(int16_t) * (size_t)cfg->G * cfg->slots_per_rank;
    CUDA_TRY(cudaMemcpyAsync(cand_stage, candidates_host, row * (size_t)P * cfg->L, cudaMemcpyHostToDevice, stream));
    int32_t* argmin_dev = argmin_host ? reinterpret_cast<int32_t*>(w.mp.bad + 32) : nullptr;
    rc = gimbal_eval_placements(cfg, P, cand_stage, A, B, D, M, M_scalar, prev, out_stage, argmin_dev, workspace, workspace_bytes, stream_);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpyAsync(out_host, out_stage, sizeof(float) * 5 * (size_t)P, cudaMemcpyDeviceToHost, stream));
    if (argmin_host) CUDA_TRY(cudaMemcpyAsync(argmin_host, argmin_dev, sizeof(int32_t), cudaMemcpyDeviceToHost, stream));
    CUDA_TRY(cudaStreamSynchronize(stream));
    return GIMBAL_OK;
}

int gimbal_eval_moves(const gimbal_placement_cfg* cfg, const int16_t* cur, const int16_t* prev, int64_t n_moves, const int32_t* moves,
                      const void* A, const void* B, const float* D, const float* M, float M_scalar, float* delta,
                      int32_t* best_per_layer, void* workspace, size_t workspace_bytes, gimbal_stream_t stream_) {
    int rc = validate_place_cfg(cfg);
    if (rc) return rc;
    if (n_moves < 0) return fail(GIMBAL_ERR_INVALID_ARG, "n_moves < 0");
    if (!cur || !prev || !A || !B || !D || (n_moves > 0 && !delta)) return fail(GIMBAL_ERR_INVALID_ARG, "NULL argument");
    const long long NS = (long long)cfg->G * cfg->slots_per_rank;
    if (!moves && n_moves != (long long)cfg->L * NS * (NS - 1) / 2)
        return fail(GIMBAL_ERR_INVALID_ARG, "implicit neighbourhood has %lld moves, got %lld", (long long)cfg->L * NS * (NS - 1) / 2, (long long)n_moves);
    if (n_moves > 0xffffffffll) return fail(GIMBAL_ERR_UNSUPPORTED, "n_moves > 2^32-1");
    PlaceWs w;
    const size_t need = place_ws_carve(cfg, 0, workspace, &w);
    if (!workspace || workspace_bytes < need) return fail(GIMBAL_ERR_WORKSPACE, "workspace %zu < %zu bytes", workspace_bytes, need);
    // the whole-neighbourhood kernel stages the layer's per-slot rows in shared memory; larger shapes take the per-move kernel
    const bool use_all = n_moves > 0 && !moves && cfg->G >= 4 && move_all_smem_bytes((int)NS, cfg->G, M != nullptr) <= kSmemLimit;
    rc = require_device();
    if (rc) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    rc = launch_tables(cfg, A, B, D, M, M_scalar, prev, w, stream);
    if (rc) return rc;
    CUDA_TRY(cudaMemsetAsync(w.mp.bad, 0, sizeof(int32_t), stream));
    MovePrepParams pp{};
    pp.L = cfg->L; pp.E = cfg->E; pp.G = cfg->G; pp.sp = cfg->slots_per_rank; pp.cur = cur; pp.t = w.t; pp.mp = w.mp;
    move_prep_kernel<<<cfg->L, 256, 0, stream>>>(pp);
    LAUNCH_CHECK("move_prep_kernel");
    if (best_per_layer) {
        fill_u64_kernel<<<(cfg->L + 255) / 256, 256, 0, stream>>>(w.best, ~0ull, cfg->L);
        LAUNCH_CHECK("fill_u64_kernel");
    }
    if (use_all) {
        // implicit neighbourhood: blocks of ~2048 pair indices of one layer, tables staged in shared memory
        MoveAllParams ap{};
        ap.L = cfg->L; ap.E = cfg->E; ap.G = cfg->G; ap.sp = cfg->slots_per_rank; ap.has_M = M != nullptr;
        ap.alpha = cfg->alpha; ap.beta = cfg->beta; ap.gamma = cfg->gamma; ap.M_scalar = M_scalar;
        ap.cur = cur; ap.t = w.t; ap.mp = w.mp; ap.delta = delta; ap.best = best_per_layer ? w.best : nullptr;
        int lg = 0;
        while ((1 << lg) < cfg->G) ++lg;
        ap.lgG = lg;
        // a warp task = the row pair {a, NS-2-a} (NS-1 moves).  One balanced wave: as many blocks per layer as give every SM
        // its three resident blocks' worth (each block stages the layer's rows once), at least one task per warp
        const int n_tasks = (int)(NS / 2);
        const size_t smem_all = move_all_smem_bytes((int)NS, cfg->G, M != nullptr);
        int per_sm = (int)((kSmemLimit - 1024) / (smem_all + 1024));
        constexpr int kMaxResident = 2048 / kMoveAllThreads / 2;          // 64 registers per thread
        per_sm = per_sm > kMaxResident ? kMaxResident : (per_sm < 1 ? 1 : per_sm);
        int bpl = per_sm * device_info().sms / cfg->L;
        const int max_bpl = (n_tasks + kMoveAllThreads / 32 - 1) / (kMoveAllThreads / 32);
        if (bpl > max_bpl) bpl = max_bpl;
        if (bpl < 1) bpl = 1;
        ap.tasks_per_block = (n_tasks + bpl - 1) / bpl;
        bpl = (n_tasks + ap.tasks_per_block - 1) / ap.tasks_per_block;
        {
            MoveSlotsParams sl{};
            sl.L = cfg->L; sl.E = cfg->E; sl.G = cfg->G; sl.sp = cfg->slots_per_rank; sl.lgG = lg; sl.has_M = ap.has_M;
            sl.cur = cur; sl.t = w.t; sl.mp = w.mp;
            move_slots_kernel<<<dim3((unsigned)((NS * cfg->G + 255) / 256), cfg->L), 256, 0, stream>>>(sl);
            LAUNCH_CHECK("move_slots_kernel");
        }
        const size_t smem = smem_all;
        auto kern = ap.has_M ? move_all_kernel<true> : move_all_kernel<false>;
        CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        ktime_begin(GIMBAL_KERNEL_MOVES, stream);
        kern<<<dim3(bpl, cfg->L), kMoveAllThreads, smem, stream>>>(ap);
        ktime_end(GIMBAL_KERNEL_MOVES, stream);
        LAUNCH_CHECK("move_all_kernel");
    } else if (n_moves > 0) {
        MoveParams mp{};
        mp.L = cfg->L; mp.E = cfg->E; mp.G = cfg->G; mp.sp = cfg->slots_per_rank; mp.n_moves = n_moves; mp.moves = moves; mp.cur = cur;
        mp.alpha = cfg->alpha; mp.beta = cfg->beta; mp.gamma = cfg->gamma; mp.M_scalar = M_scalar; mp.has_M = M != nullptr;
        mp.t = w.t; mp.mp = w.mp; mp.delta = delta; mp.best = best_per_layer ? w.best : nullptr;
        const long long blocks = (n_moves + 255) / 256;
        ktime_begin(GIMBAL_KERNEL_MOVES, stream);
        move_delta_kernel<<<(unsigned)blocks, 256, 0, stream>>>(mp);
        ktime_end(GIMBAL_KERNEL_MOVES, stream);
        LAUNCH_CHECK("move_delta_kernel");
    }
    if (best_per_layer) {
        best_to_index_kernel<<<(cfg->L + 255) / 256, 256, 0, stream>>>(w.best, best_per_layer, cfg->L);
        LAUNCH_CHECK("best_to_index_kernel");
    }
    return GIMBAL_OK;
}

int gimbal_eval_moves_host(const gimbal_placement_cfg* cfg, const int16_t* cur_host, const int16_t* prev_host, int16_t* cur_stage,
                           int16_t* prev_stage, int64_t n_moves, const int32_t* moves_host, int32_t* moves_stage, const void* A,
                           const void* B, const float* D, const float* M, float M_scalar, float* delta_stage, float* delta_host,
                           int32_t* best_stage, int32_t* best_host, void* workspace, size_t workspace_bytes, gimbal_stream_t stream_) {
    int rc = validate_place_cfg(cfg);
    if (rc) return rc;
    if (n_moves < 0) return fail(GIMBAL_ERR_INVALID_ARG, "n_moves < 0");
    if (!cur_host || !prev_host || !cur_stage || !prev_stage || (n_moves > 0 && !delta_stage) || (moves_host && !moves_stage) ||
        (best_host && !best_stage))
        return fail(GIMBAL_ERR_INVALID_ARG, "NULL host / staging pointer");
    rc = require_device();
    if (rc) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const size_t nb = sizeof(int16_t) * (size_t)cfg->L * cfg->G * cfg->slots_per_rank;
    CUDA_TRY(cudaMemcpyAsync(cur_stage, cur_host, nb, cudaMemcpyHostToDevice, stream));
    CUDA_TRY(cudaMemcpyAsync(prev_stage, prev_host, nb, cudaMemcpyHostToDevice, stream));
    if (moves_host && n_moves > 0) CUDA_TRY(cudaMemcpyAsync(moves_stage, moves_host, sizeof(int32_t) * 3 * (size_t)n_moves, cudaMemcpyHostToDevice, stream));
    rc = gimbal_eval_moves(cfg, cur_stage, prev_stage, n_moves, moves_host ? moves_stage : nullptr, A, B, D, M, M_scalar, delta_stage,
                           best_host ? best_stage : nullptr, workspace, workspace_bytes, stream_);
    if (rc) return rc;
    if (delta_host && n_moves > 0) CUDA_TRY(cudaMemcpyAsync(delta_host, delta_stage, sizeof(float) * 5 * (size_t)n_moves, cudaMemcpyDeviceToHost, stream));
    if (best_host) CUDA_TRY(cudaMemcpyAsync(best_host, best_stage, sizeof(int32_t) * cfg->L, cudaMemcpyDeviceToHost, stream));
    CUDA_TRY(cudaStreamSynchronize(stream));
    return GIMBAL_OK;
}

int gimbal_refine_placement(const gimbal_placement_cfg* cfg, int16_t* cur, const int16_t* prev, int iters, const void* A, const void* B,
                            const float* D, const float* M, float M_scalar, float* delta, int32_t* best, int32_t* applied,
                            void* workspace, size_t workspace_bytes, gimbal_stream_t stream_) {
    int rc = validate_place_cfg(cfg);
    if (rc) return rc;
    if (iters < 0 || !best || !delta) return fail(GIMBAL_ERR_INVALID_ARG, "iters < 0 or NULL scratch");
    const long long NS = (long long)cfg->G * cfg->slots_per_rank;
    const long long n = (long long)cfg->L * NS * (NS - 1) / 2;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    if (applied) {
        rc = require_device();
        if (rc) return rc;
        CUDA_TRY(cudaMemsetAsync(applied, 0, sizeof(int32_t) * cfg->L, stream));
    }
    for (int it = 0; it < iters; ++it) {
        rc = gimbal_eval_moves(cfg, cur, prev, n, nullptr, A, B, D, M, M_scalar, delta, best, workspace, workspace_bytes, stream_);
        if (rc) return rc;
        apply_best_moves_kernel<<<(cfg->L + 127) / 128, 128, 0, stream>>>(cfg->L, (int)NS, cfg->alpha, cfg->beta, cfg->gamma, best, delta, cur, applied);
        LAUNCH_CHECK("apply_best_moves_kernel");
    }
    return GIMBAL_OK;
}

int gimbal_build_expert_map(int L, int E, int G, int slots_per_rank, const int16_t* placement, int32_t* rep_off, int16_t* rep_slots,
                            int32_t* status, gimbal_stream_t stream_) {
    if (L < 1 || E < 1 || E > kMaxE || G < 1 || G > kMaxG || slots_per_rank < 1 || slots_per_rank > 16)
        return fail(GIMBAL_ERR_INVALID_ARG, "expert map: L >= 1, 1 <= E <= %d, 1 <= G <= %d, 1 <= slots_per_rank <= 16", kMaxE, kMaxG);
    if (!placement || !rep_off || !rep_slots) return fail(GIMBAL_ERR_INVALID_ARG, "NULL argument");
    int rc = require_device();
    if (rc) return rc;
    expert_map_kernel<<<L, 256, 0, static_cast<cudaStream_t>(stream_)>>>(E, G * slots_per_rank, placement, rep_off, rep_slots, status);
    LAUNCH_CHECK("expert_map_kernel");
    return GIMBAL_OK;
}

int gimbal_greedy_place(const gimbal_placement_cfg* cfg, const void* A, const void* B, const float* D, const float* M, float M_scalar,
                        const int16_t* prev, int16_t* out, int32_t* status, gimbal_stream_t stream_) {
    int rc = validate_place_cfg(cfg);
    if (rc) return rc;
    if (!A || !B || !D || !prev || !out) return fail(GIMBAL_ERR_INVALID_ARG, "NULL argument");
    const int NS = cfg->G * cfg->slots_per_rank;
    const size_t smem = greedy_smem_bytes(cfg->E, cfg->G, NS);
    if (smem > kSmemLimit) return fail(GIMBAL_ERR_UNSUPPORTED, "greedy placement: E=%d G=%d needs %zu B of shared memory", cfg->E, cfg->G, smem);
    rc = require_device();
    if (rc) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    GreedyParams gp{};
    gp.L = cfg->L; gp.E = cfg->E; gp.G = cfg->G; gp.sp = cfg->slots_per_rank; gp.S = cfg->S;
    gp.counts_f32 = cfg->counts_dtype == GIMBAL_COUNTS_F32;
    gp.A = A; gp.B = B; gp.D = D; gp.M = M; gp.M_scalar = M_scalar;
    gp.alpha = cfg->alpha; gp.beta = cfg->beta; gp.gamma = cfg->gamma; gp.prev = prev; gp.out = out; gp.status = status;
    CUDA_TRY(cudaFuncSetAttribute(greedy_place_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ktime_begin(GIMBAL_KERNEL_GREEDY, stream);
    greedy_place_kernel<<<cfg->L, kGreedyThreads, smem, stream>>>(gp);
    ktime_end(GIMBAL_KERNEL_GREEDY, stream);
    LAUNCH_CHECK("greedy_place_kernel");
    return GIMBAL_OK;
}

int gimbal_select_engines(const gimbal_sched_cfg* cfg, int B, const float* trace, const uint8_t* complete, const float* req_len,
                          double* comp, int32_t* rr, int32_t* engine, gimbal_stream_t stream_) {
    if (!cfg) return fail(GIMBAL_ERR_INVALID_ARG, "cfg is NULL");
    if (cfg->N < 1 || cfg->N > 64 || cfg->R < 0 || B < 0) return fail(GIMBAL_ERR_INVALID_ARG, "need 1 <= N <= 64, R >= 0, B >= 0");
    if (B > 0 && (!trace || !comp || !rr || (cfg->R > 0 && (!req_len || !engine)))) return fail(GIMBAL_ERR_INVALID_ARG, "NULL argument");
    if (reinterpret_cast<uintptr_t>(trace) & 15) return fail(GIMBAL_ERR_INVALID_ARG, "trace must be 16-byte aligned");
    int rc = require_device();
    if (rc) return rc;
    if (B == 0) return GIMBAL_OK;
    SchedParams sp{};
    sp.B = B; sp.N = cfg->N; sp.R = cfg->R;
    sp.high_kv = cfg->high_kv; sp.large_gap = cfg->large_gap; sp.lambda_kv = cfg->lambda_kv; sp.lambda_moe = cfg->lambda_moe;
    sp.close_frac = cfg->close_frac;
    sp.trace = trace; sp.complete = complete; sp.req_len = req_len; sp.comp = comp; sp.rr = rr; sp.engine = engine;
    select_engines_kernel<<<(B + kSchedWarps - 1) / kSchedWarps, kSchedWarps * 32, 0, static_cast<cudaStream_t>(stream_)>>>(sp);
    LAUNCH_CHECK("select_engines_kernel");
    return GIMBAL_OK;
}

int gimbal_order_queues(int B, int Q, const float* arrival, const int32_t* prefill, const int32_t* qlen, float now, float theta_age,
                        int32_t* order, gimbal_stream_t stream_) {
    if (B < 0 || Q < 1 || Q > kQueueMax) return fail(GIMBAL_ERR_INVALID_ARG, "need B >= 0 and 1 <= Q <= %d", kQueueMax);
    if (B > 0 && (!arrival || !prefill || !qlen || !order)) return fail(GIMBAL_ERR_INVALID_ARG, "NULL argument");
    int rc = require_device();
    if (rc) return rc;
    if (B == 0) return GIMBAL_OK;
    QueueParams qp{B, Q, now, theta_age, arrival, prefill, qlen, order};
    order_queues_kernel<<<B, kQueueThreads, 0, static_cast<cudaStream_t>(stream_)>>>(qp);
    LAUNCH_CHECK("order_queues_kernel");
    return GIMBAL_OK;
}

}  // extern "C"
