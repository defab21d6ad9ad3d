// a4 + a5: window / EMA update of the [L,S,E] profile, per-expert load B and per-source MoE
// pressure (R2, R14).  One block per layer, thread
// e owns expert e; the last block to finish reduces the per-layer pressure partials in layer
// order (deterministic) and advances the device-side step counter.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gimbal {

struct UpdateParams {
    int L, S, E, G, sp;
    int mode, window_len;
    float ema_decay;
    const int32_t* A_step;
    int32_t* A_win; int32_t* A_pub; int32_t* B_pub;
    float* A_ema;
    void* B;
    float* pressure_raw; float* pressure_rel;
    int64_t* step_counter;
    int32_t* status;
    const int16_t* cur_placement;   // [L,NS] | nullptr
    const int32_t* dp_of_rank;      // [G] | nullptr
    double* partial;                // workspace [L,S]
    unsigned int* done_counter;     // workspace, zero on entry, reset on exit
};

constexpr int kUpdateThreads = 256;

constexpr int kUpdatePartStage = 2048;

// scratch of one layer's update: [E <= 256] live B, [E] replica counts, [G <= 64] rank loads, two flags
struct UpdateScratch {
    double b[256];
    int r[256];
    double lg[64];
    int dp[64];
    int bad;
    int last;
    double part[kUpdatePartStage];      // the [L][S] pressure partials, staged for the final reduction
};

// a4 + a5 of ONE layer by `nthr` threads (tid 0..nthr-1) that can synchronise through `sync()`; `done_counter` counts the layers
// of the step: the caller that finishes the L-th layer reduces the pressure partials over layers in fixed order (deterministic),
// advances the step counter and leaves the counter at 0.  Used by stats_update_kernel (one block per layer) and by the fused
// router kernel in the one-tile-per-layer regime (the CTA pair that owns the layer's complete histogram).
// `step` = *p.step_counter read by the caller (as early as its ordering allows); `a_step(s, e)` = this layer's fresh counts (global
// A_step for the kernel below, the router kernel's own shared-memory histogram in its tail).
template <class Sync, class Counts>
__device__ __forceinline__ void stats_update_layer(const UpdateParams& p, int l, int tid, int nthr, UpdateScratch& sh, int64_t step, Sync sync,
                                                   Counts a_step) {
    const bool publish = p.mode == 0 && ((step + 1) % p.window_len) == 0;
    if (tid == 0) { sh.bad = 0; sh.last = 0; }
    for (int e = tid; e < 256; e += nthr) sh.r[e] = 0;
    const bool want_pressure = p.cur_placement != nullptr && p.dp_of_rank != nullptr;
    if (want_pressure)
        for (int g = tid; g < p.G; g += nthr) sh.dp[g] = p.dp_of_rank[g];
    sync();

    for (int e = tid; e < p.E; e += nthr) {
        // sources are read sixteen at a time before anything is written back: the loads of a batch are in
        // flight together instead of one global round trip per source
        if (p.mode == 0) {
            int64_t b = 0;
            for (int s0 = 0; s0 < p.S; s0 += 16) {
                int32_t win[16], stp[16];
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const int sj = min(s0 + j, p.S - 1);
                    win[j] = p.A_win[((size_t)l * p.S + sj) * p.E + e]; stp[j] = a_step(sj, e);
                }
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    if (s0 + j < p.S) {
                        const size_t i = ((size_t)l * p.S + s0 + j) * p.E + e;
                        const int64_t w = (int64_t)win[j] + stp[j];
                        if (w > INT32_MAX) sh.bad = 1;       // window sum must fit int32
                        b += w;
                        if (publish) { p.A_pub[i] = (int32_t)w; p.A_win[i] = 0; }
                        else p.A_win[i] = (int32_t)w;
                    }
                }
            }
            if (b > INT32_MAX) sh.bad = 1;
            reinterpret_cast<int32_t*>(p.B)[(size_t)l * p.E + e] = (int32_t)b;
            if (publish) p.B_pub[(size_t)l * p.E + e] = (int32_t)b;
            sh.b[e] = (double)b;
        } else {
            float b = 0.0f;
            for (int s0 = 0; s0 < p.S; s0 += 16) {
                float ema[16]; int32_t stp[16];
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const int sj = min(s0 + j, p.S - 1);
                    ema[j] = p.A_ema[((size_t)l * p.S + sj) * p.E + e]; stp[j] = a_step(sj, e);
                }
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    if (s0 + j < p.S) {
                        const float a = __fmaf_rn(p.ema_decay, ema[j], (float)stp[j]);
                        p.A_ema[((size_t)l * p.S + s0 + j) * p.E + e] = a;
                        b = __fadd_rn(b, a);
                    }
                }
            }
            reinterpret_cast<float*>(p.B)[(size_t)l * p.E + e] = b;
            sh.b[e] = (double)b;
        }
    }

    if (want_pressure) {
        const int NS = p.G * p.sp;
        const int16_t* pl = p.cur_placement + (size_t)l * NS;
        for (int j = tid; j < NS; j += nthr) {
            const int x = pl[j];
            if (x < 0 || x >= p.E) sh.bad = 1; else atomicAdd(&sh.r[x], 1);
        }
        sync();
        for (int g = tid; g < p.G; g += nthr) {
            double lg = 0.0;
            for (int j = 0; j < p.sp; ++j) {
                const int x = pl[g * p.sp + j];
                if (x >= 0 && x < p.E) lg += sh.b[x] / (double)sh.r[x];
            }
            sh.lg[g] = lg;
        }
        sync();
        for (int s = tid; s < p.S; s += nthr) {
            double acc = 0.0;
            for (int g = 0; g < p.G; ++g)
                if (sh.dp[g] == s) acc += sh.lg[g];
            p.partial[(size_t)l * p.S + s] = acc;
        }
    }
    sync();
    if (tid == 0 && sh.bad && p.status) atomicOr(p.status, 1);

    // last layer of the step: deterministic reduction over layers, then advance the step counter
    __threadfence();
    sync();
    if (tid == 0) sh.last = (atomicAdd(p.done_counter, 1u) == (unsigned)p.L - 1u);
    sync();
    if (sh.last) {
        __threadfence();
        if (want_pressure) {
            // every thread fetches its share of the [L][S] partials at once (one round trip instead of L dependent ones), then source
            // s adds its column in layer order -- the same order, hence the same doubles, as a plain loop over the layers
            const int n = p.L * p.S;
            const bool staged = n <= kUpdatePartStage;
            if (staged) {
                for (int i = tid; i < n; i += nthr) sh.part[i] = __ldcg(p.partial + i);
                sync();
            }
            for (int s = tid; s < p.S; s += nthr) {
                double acc = 0.0;
                for (int ll = 0; ll < p.L; ++ll) acc += staged ? sh.part[ll * p.S + s] : __ldcg(p.partial + (size_t)ll * p.S + s);
                sh.lg[s] = acc;
            }
        }
        sync();
        if (want_pressure) {
            for (int s = tid; s < p.S; s += nthr) {
                double tot = 0.0;
                for (int q = 0; q < p.S; ++q) tot += sh.lg[q];
                p.pressure_raw[s] = (float)sh.lg[s];
                p.pressure_rel[s] = tot > 0.0 ? (float)(sh.lg[s] * p.S / tot) : 1.0f;
            }
        }
        if (tid == 0) {
            *p.step_counter = step + 1;
            *p.done_counter = 0u;
        }
    }
}

#ifdef GIMBAL_DEFINE_STATS_UPDATE_KERNEL        // the kernel itself lives in one translation unit (gimbal_api.cu)
__global__ void __launch_bounds__(kUpdateThreads) stats_update_kernel(const UpdateParams p) {
    __shared__ UpdateScratch sh;
    // programmatic dependent launch: this grid may have been scheduled while the router kernel still ran -- wait for it (and its
    // memory) here; the next kernel of the stream may be scheduled from now on (it waits for this grid before it writes A_step)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int l = blockIdx.x;
    const int32_t* a = p.A_step + (size_t)l * p.S * p.E;
    const int E = p.E;
    stats_update_layer(p, l, threadIdx.x, kUpdateThreads, sh, *p.step_counter, [] { __syncthreads(); },
                       [a, E](int s, int e) { return a[(size_t)s * E + e]; });
}
#endif

}  // namespace gimbal
