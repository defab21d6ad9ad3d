// Host-side helpers shared by the translation units of libgimbal (error reporting, device
// probe, TMA descriptor encoding, launch arguments).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/gimbal.h"
#include "gating.cuh"
#include "stats_update.cuh"

namespace gimbal {

int fail(int code, const char* fmt, ...);
void count_launch();
// optional CUDA-event brackets around the main kernels (gimbal_kernel_timing)
void ktime_begin(int which, cudaStream_t s);
void ktime_end(int which, cudaStream_t s);

#define CUDA_TRY(expr)                                                                         \
    do {                                                                                       \
        cudaError_t _e = (expr);                                                               \
        if (_e != cudaSuccess) return ::gimbal::fail(GIMBAL_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(_e)); \
    } while (0)

#define LAUNCH_CHECK(name)                                                                     \
    do {                                                                                       \
        ::gimbal::count_launch();                                                              \
        cudaError_t _e = cudaGetLastError();                                                   \
        if (_e != cudaSuccess) return ::gimbal::fail(GIMBAL_ERR_CUDA, "launch %s: %s", name, cudaGetErrorString(_e)); \
    } while (0)

struct DeviceInfo {
    bool ok = false;
    int sms = 0;
    char why[128] = "";
};
const DeviceInfo& device_info();
int require_device();

constexpr size_t kSmemLimit = 227 * 1024;

// bf16 tensor [d2][d1][d0] (d0 contiguous), box [1][box1][64], 128-byte swizzle
int make_tmap_bf16_3d(CUtensorMap* m, const void* ptr, uint64_t d0, uint64_t d1, uint64_t d2, uint32_t box1);

int make_tmap_rows_i16_4d(CUtensorMap* m, const void* ptr, uint32_t piece, uint32_t npieces, uint64_t L, uint64_t P, uint32_t box0,
                          uint32_t boxP);

struct RouteArgs {
    const gimbal_router_cfg* cfg;
    int layer0, n_layers, T;
    const void* hidden; const void* w_router;
    const float* select_bias; const float* src_logit_bias; const int32_t* src_offsets;
    float* logits; int32_t* topk_ids; float* topk_w;
    int32_t* A_step;
    unsigned int* zero_word;   // | nullptr: workspace word the fused router kernel clears (saves a memset node per step)
    const int32_t* rep_off; const int16_t* rep_slots; int32_t* phys_ids; int map_NS;   // expert mapping | nullptr
    int fuse_gate;
    int cta_group;          // 1 or 2
    int hist_agg;           // epilogue counts by columns (GIMBAL_OPT_HIST_AGG)
    const UpdateParams* upd; // | nullptr: the router kernel runs the window / EMA update of the layers it stores (whole-step call, one tile per layer)
    int pdl;                // programmatic dependent launch of the router kernel / stats_update_kernel (GIMBAL_OPT_PDL)
    int store_hist;         // the caller skipped the zeroing of A_step: every layer is one tile with its own CTA (pair)
    int epi_parts;          // 1 or 2 epilogue warps per TMEM lane quadrant (GIMBAL_OPT_EPI_PARTS; 2 only takes effect for E >= 128, counts only)
    cudaStream_t stream;
};

GateParams gate_params(const gimbal_router_cfg* c);

// one translation unit per expert count (route_e*.cu)
#define GIMBAL_DECL_E(E) int launch_gemm_e##E(const RouteArgs& a); int launch_gate_e##E(const RouteArgs& a);
GIMBAL_DECL_E(16) GIMBAL_DECL_E(32) GIMBAL_DECL_E(64) GIMBAL_DECL_E(128) GIMBAL_DECL_E(256)
#undef GIMBAL_DECL_E

}  // namespace gimbal
