// Definitions of host_common.h.
#include "host_common.h"

#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <mutex>

namespace gimbal {

static std::mutex g_err_mu;
static char g_err[512] = "";
static std::atomic<int64_t> g_launches{0};

int fail(int code, const char* fmt, ...) {
    std::lock_guard<std::mutex> lk(g_err_mu);
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

static bool g_ktime_on = false;
constexpr int kTimedKernels = 8;
static cudaEvent_t g_kev[kTimedKernels][2];
static bool g_kev_made = false, g_kev_rec[kTimedKernels] = {};
int ktime_enable(int on) {
    if (on && !g_kev_made) {
        for (int i = 0; i < kTimedKernels; ++i)
            for (int j = 0; j < 2; ++j)
                if (cudaEventCreate(&g_kev[i][j]) != cudaSuccess) return fail(GIMBAL_ERR_CUDA, "cudaEventCreate failed");
        g_kev_made = true;
    }
    g_ktime_on = on != 0;
    return GIMBAL_OK;
}
void ktime_begin(int which, cudaStream_t s) { if (g_ktime_on) cudaEventRecord(g_kev[which][0], s); }
void ktime_end(int which, cudaStream_t s) { if (g_ktime_on) { cudaEventRecord(g_kev[which][1], s); g_kev_rec[which] = true; } }
int ktime_elapsed(int which, float* ms) {
    if (which < 0 || which >= kTimedKernels || !ms) return fail(GIMBAL_ERR_INVALID_ARG, "kernel id %d", which);
    if (!g_kev_made || !g_kev_rec[which]) return fail(GIMBAL_ERR_INVALID_ARG, "kernel %d was not timed", which);
    if (cudaEventSynchronize(g_kev[which][1]) != cudaSuccess) return fail(GIMBAL_ERR_CUDA, "cudaEventSynchronize failed");
    if (cudaEventElapsedTime(ms, g_kev[which][0], g_kev[which][1]) != cudaSuccess) return fail(GIMBAL_ERR_CUDA, "cudaEventElapsedTime failed");
    return GIMBAL_OK;
}
int64_t launches() { return g_launches.load(); }
void copy_last_error(char* buf, size_t n) {
    std::lock_guard<std::mutex> lk(g_err_mu);
    snprintf(buf, n, "%s", g_err);
}

// One record per device ordinal, filled on the first call made with that device current: a process that drives several
// GPUs gets each one's SM count (grid sizes follow it), not the count of whichever device came first.
const DeviceInfo& device_info() {
    constexpr int kMaxDevices = 64;
    static DeviceInfo info[kMaxDevices];
    static std::atomic<int> state[kMaxDevices];          // 0 = not probed, 2 = ready
    static std::mutex mu;
    static DeviceInfo none = [] { DeviceInfo d; snprintf(d.why, sizeof d.why, "no CUDA device"); return d; }();
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
        cudaGetLastError();
        return none;
    }
    if (state[dev].load(std::memory_order_acquire) == 2) return info[dev];
    std::lock_guard<std::mutex> lk(mu);
    if (state[dev].load(std::memory_order_relaxed) != 2) {
        DeviceInfo d;
        int major = 0;
        cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev);
        if (major != 10) snprintf(d.why, sizeof d.why, "device %d: compute capability %d.x, need 10.x (sm_100a)", dev, major);
        else d.ok = true;
        info[dev] = d;
        state[dev].store(2, std::memory_order_release);
    }
    return info[dev];
}

int require_device() {
    const DeviceInfo& d = device_info();
    if (!d.ok) return fail(GIMBAL_ERR_UNSUPPORTED, "%s", d.why);
    return GIMBAL_OK;
}

// ---- TMA descriptors -----------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = [] {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess) f = nullptr;
        return reinterpret_cast<EncodeTiledFn>(f);
    }();
    return fn;
}

// bf16 tensor [d2][d1][d0] (d0 contiguous), box [1][box1][64], 128-byte swizzle
int make_tmap_bf16_3d(CUtensorMap* m, const void* ptr, uint64_t d0, uint64_t d1, uint64_t d2, uint32_t box1) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return fail(GIMBAL_ERR_CUDA, "cuTensorMapEncodeTiled not available");
    cuuint64_t dims[3] = {d0, d1, d2};
    cuuint64_t strides[2] = {d0 * 2, d0 * d1 * 2};
    cuuint32_t box[3] = {64, box1, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(ptr), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(GIMBAL_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
    return GIMBAL_OK;
}

// candidate rows [P][L][NS] int16 seen as [P][L][NS/piece][piece]; the box is `box0` >= piece elements wide, so every piece
// lands at a pitch of box0 elements in shared memory with the tail zero-filled (out-of-bounds fill), `boxP` candidates per copy
int make_tmap_rows_i16_4d(CUtensorMap* m, const void* ptr, uint32_t piece, uint32_t npieces, uint64_t L, uint64_t P, uint32_t box0,
                          uint32_t boxP) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return fail(GIMBAL_ERR_CUDA, "cuTensorMapEncodeTiled not available");
    cuuint64_t dims[4] = {piece, npieces, L, P};
    cuuint64_t strides[3] = {(cuuint64_t)piece * 2, (cuuint64_t)piece * npieces * 2, (cuuint64_t)piece * npieces * 2 * L};
    cuuint32_t box[4] = {box0, npieces, 1, boxP};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_UINT16, 4, const_cast<void*>(ptr), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(GIMBAL_ERR_CUDA, "cuTensorMapEncodeTiled (candidate rows) failed (%d)", (int)r);
    return GIMBAL_OK;
}

GateParams gate_params(const gimbal_router_cfg* c) {
    GateParams g;
    g.k = c->k; g.score_fn = c->score_fn; g.renorm = c->renorm; g.n_groups = c->n_groups;
    g.topk_groups = c->topk_groups; g.topn = c->group_score_topn; g.routed_scale = c->routed_scale;
    return g;
}


}  // namespace gimbal
