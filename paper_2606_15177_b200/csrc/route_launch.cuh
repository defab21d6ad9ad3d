// Launchers of the router GEMM and the standalone gating kernel, instantiated once per
// expert count in route_e*.cu so that the translation units compile in parallel.
#pragma once
#include "host_common.h"
#include "router_gemm.cuh"

namespace gimbal {

template <int N, int kCG, bool kSig, int kEP = 1>
int launch_gemm_t(const RouteArgs& a) {
    const gimbal_router_cfg* c = a.cfg;
    CUtensorMap ta, tb;
    int rc = make_tmap_bf16_3d(&ta, a.hidden, (uint64_t)c->H, (uint64_t)a.T, (uint64_t)a.n_layers, kBlockM);
    if (rc) return rc;
    rc = make_tmap_bf16_3d(&tb, a.w_router, (uint64_t)c->H, (uint64_t)c->E, (uint64_t)c->L, N / kCG);
    if (rc) return rc;
    GemmParams p{};
    p.n_layers = a.n_layers; p.layer0 = a.layer0; p.T = a.T; p.H = c->H; p.S = c->S;
    p.m_tiles = (a.T + kBlockM * kCG - 1) / (kBlockM * kCG);
    const bool out = a.fuse_gate && (a.topk_ids || a.topk_w || a.rep_off);
    p.stages = gemm_pick_stages<N, kCG>(c->S, out, kEP);
    p.hist_agg = a.hist_agg;
    if (p.stages < 2) return fail(GIMBAL_ERR_UNSUPPORTED, "router GEMM: not enough shared memory for E=%d S=%d", N, c->S);
    p.src_logit_bias = a.src_logit_bias; p.src_offsets = a.src_offsets; p.logits = a.logits;
    p.do_gate = a.fuse_gate; p.select_bias = a.select_bias; p.topk_ids = a.topk_ids; p.topk_w = a.topk_w;
    p.A_step = a.A_step; p.gp = gate_params(c); p.zero_word = a.zero_word;
    p.map = ExpertMap{a.rep_off, a.rep_slots, a.phys_ids, a.map_NS};
    const size_t smem = gemm_smem_bytes<N, kCG>(c->S, p.stages, out, kEP);
    auto kern = router_gemm_kernel<N, kCG, kSig, kEP>;
    CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int sms = device_info().sms;
    const int n_tiles = p.n_layers * p.m_tiles;
    int pairs = sms / kCG;
    if (pairs > n_tiles) pairs = n_tiles;
    p.store_hist = a.store_hist && a.fuse_gate && p.m_tiles == 1 && n_tiles <= sms / kCG;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(pairs * kCG);
    cfg.blockDim = dim3(128 + 128 * kEP);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = a.stream;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = kCG; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    p.pdl = p.store_hist ? a.pdl : 0;
    p.fuse_update = p.store_hist && a.upd != nullptr;
    if (p.fuse_update) p.upd = *a.upd;
    cfg.attrs = attr; cfg.numAttrs = p.pdl ? 2 : 1;
    ktime_begin(GIMBAL_KERNEL_ROUTER, a.stream);
    CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, ta, tb, p));
    ktime_end(GIMBAL_KERNEL_ROUTER, a.stream);
    LAUNCH_CHECK("router_gemm_kernel");
    return GIMBAL_OK;
}

template <int N>
int launch_gemm_n(const RouteArgs& a) {
    const bool sig = a.cfg->score_fn == GIMBAL_SCORE_SIGMOID;
    if constexpr (N >= 128) {
        // two epilogue warps per TMEM lane quadrant (each half of the experts) where the epilogue is exposed: counts only and at
        // most two tiles per CTA (pair) -- the small-batch regime, one 128 / 256-token tile per layer
        if (a.epi_parts == 2 && a.fuse_gate && !a.logits && !a.topk_ids && !a.topk_w && !a.rep_off) {
            if (a.cta_group == 2) return sig ? launch_gemm_t<N, 2, true, 2>(a) : launch_gemm_t<N, 2, false, 2>(a);
            return sig ? launch_gemm_t<N, 1, true, 2>(a) : launch_gemm_t<N, 1, false, 2>(a);
        }
    }
    if (a.cta_group == 2) return sig ? launch_gemm_t<N, 2, true>(a) : launch_gemm_t<N, 2, false>(a);
    return sig ? launch_gemm_t<N, 1, true>(a) : launch_gemm_t<N, 1, false>(a);
}


// ---- standalone gating ---------------------------------------------------------------------
template <int E, bool kSig, bool kOut>
int launch_gate_v(const GateKernelParams& p, dim3 grid, int S, cudaStream_t stream) {
    const size_t smem = gate_smem_bytes<E, kOut>(S);
    if (smem > kSmemLimit) return fail(GIMBAL_ERR_UNSUPPORTED, "gating: E=%d S=%d needs %zu B of shared memory", E, S, smem);
    auto kern = gate_hist_kernel<E, kSig, kOut>;
    CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<grid, gate_warps<E, kOut>() * 32, smem, stream>>>(p);
    return GIMBAL_OK;
}

template <int E>
int launch_gate_t(const RouteArgs& a) {
    GateKernelParams p{};
    p.logits = a.logits; p.select_bias = a.select_bias; p.src_offsets = a.src_offsets;
    p.topk_ids = a.topk_ids; p.topk_w = a.topk_w; p.A_step = a.A_step;
    p.layer0 = a.layer0; p.T = a.T; p.S = a.cfg->S; p.gp = gate_params(a.cfg);
    p.map = ExpertMap{a.rep_off, a.rep_slots, a.phys_ids, a.map_NS};
    dim3 grid((a.T + kGateRowsPerBlock - 1) / kGateRowsPerBlock, a.n_layers);
    const bool sig = a.cfg->score_fn == GIMBAL_SCORE_SIGMOID, out = a.topk_ids || a.topk_w || a.rep_off;
    ktime_begin(GIMBAL_KERNEL_GATE, a.stream);
    int rc;
    if (sig) rc = out ? launch_gate_v<E, true, true>(p, grid, a.cfg->S, a.stream) : launch_gate_v<E, true, false>(p, grid, a.cfg->S, a.stream);
    else rc = out ? launch_gate_v<E, false, true>(p, grid, a.cfg->S, a.stream) : launch_gate_v<E, false, false>(p, grid, a.cfg->S, a.stream);
    if (rc) return rc;
    ktime_end(GIMBAL_KERNEL_GATE, a.stream);
    LAUNCH_CHECK("gate_hist_kernel");
    return GIMBAL_OK;
}

#define GIMBAL_DEFINE_E(E)                                                     \
    int launch_gemm_e##E(const RouteArgs& a) { return launch_gemm_n<E>(a); }   \
    int launch_gate_e##E(const RouteArgs& a) { return launch_gate_t<E>(a); }

}  // namespace gimbal
