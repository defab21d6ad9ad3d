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

__global__ void __launch_bounds__(kUpdateThreads) stats_update_kernel(const UpdateParams p) {
    __shared__ double b_s[256];          // live B of this layer (E <= 256)
    __shared__ int r_s[256];             // replica count of each expert in cur_placement
    __shared__ double lg_s[64];          // rank loads (G <= 64)
    __shared__ int bad_s;
    __shared__ bool last_s;

    const int l = blockIdx.x, e = threadIdx.x;
    // programmatic dependent launch: this grid may have been scheduled while the router kernel still ran -- wait for it (and its
    // memory) here; the next kernel of the stream may be scheduled from now on (it waits for this grid before it writes A_step)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int64_t step = *p.step_counter;
    const bool publish = p.mode == 0 && ((step + 1) % p.window_len) == 0;
    if (e == 0) bad_s = 0;
    if (e < 256) r_s[e] = 0;
    __syncthreads();

    if (e < p.E) {
        // sources are read eight at a time before anything is written back: the loads of a batch are in
        // flight together instead of one global round trip per source
        if (p.mode == 0) {
            int64_t b = 0;
            for (int s0 = 0; s0 < p.S; s0 += 8) {
                int32_t win[8], stp[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const size_t i = ((size_t)l * p.S + min(s0 + j, p.S - 1)) * p.E + e;
                    win[j] = p.A_win[i]; stp[j] = p.A_step[i];
                }
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    if (s0 + j < p.S) {
                        const size_t i = ((size_t)l * p.S + s0 + j) * p.E + e;
                        const int64_t w = (int64_t)win[j] + stp[j];
                        if (w > INT32_MAX) bad_s = 1;        // window sum must fit int32
                        b += w;
                        if (publish) { p.A_pub[i] = (int32_t)w; p.A_win[i] = 0; }
                        else p.A_win[i] = (int32_t)w;
                    }
                }
            }
            if (b > INT32_MAX) bad_s = 1;
            reinterpret_cast<int32_t*>(p.B)[(size_t)l * p.E + e] = (int32_t)b;
            if (publish) p.B_pub[(size_t)l * p.E + e] = (int32_t)b;
            b_s[e] = (double)b;
        } else {
            float b = 0.0f;
            for (int s0 = 0; s0 < p.S; s0 += 8) {
                float ema[8]; int32_t stp[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const size_t i = ((size_t)l * p.S + min(s0 + j, p.S - 1)) * p.E + e;
                    ema[j] = p.A_ema[i]; stp[j] = p.A_step[i];
                }
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    if (s0 + j < p.S) {
                        const float a = __fmaf_rn(p.ema_decay, ema[j], (float)stp[j]);
                        p.A_ema[((size_t)l * p.S + s0 + j) * p.E + e] = a;
                        b = __fadd_rn(b, a);
                    }
                }
            }
            reinterpret_cast<float*>(p.B)[(size_t)l * p.E + e] = b;
            b_s[e] = (double)b;
        }
    }

    const bool want_pressure = p.cur_placement != nullptr && p.dp_of_rank != nullptr;
    if (want_pressure) {
        const int NS = p.G * p.sp;
        const int16_t* pl = p.cur_placement + (size_t)l * NS;
        for (int j = e; j < NS; j += kUpdateThreads) {
            const int x = pl[j];
            if (x < 0 || x >= p.E) bad_s = 1; else atomicAdd(&r_s[x], 1);
        }
        __syncthreads();
        if (e < p.G) {
            double lg = 0.0;
            for (int j = 0; j < p.sp; ++j) {
                const int x = pl[e * p.sp + j];
                if (x >= 0 && x < p.E) lg += b_s[x] / (double)r_s[x];
            }
            lg_s[e] = lg;
        }
        __syncthreads();
        if (e < p.S) {
            double acc = 0.0;
            for (int g = 0; g < p.G; ++g)
                if (p.dp_of_rank[g] == e) acc += lg_s[g];
            p.partial[(size_t)l * p.S + e] = acc;
        }
    }
    __syncthreads();
    if (e == 0 && bad_s && p.status) atomicOr(p.status, 1);

    // last block: deterministic reduction over layers, then advance the step counter
    __threadfence();
    __syncthreads();
    if (e == 0) last_s = (atomicAdd(p.done_counter, 1u) == (unsigned)p.L - 1u);
    __syncthreads();
    if (last_s) {
        __threadfence();
        if (want_pressure && e < p.S) {
            double acc = 0.0;
            for (int ll = 0; ll < p.L; ++ll) acc += __ldcg(p.partial + (size_t)ll * p.S + e);
            lg_s[e] = acc;
        }
        __syncthreads();
        if (want_pressure && e < p.S) {
            double tot = 0.0;
            for (int s = 0; s < p.S; ++s) tot += lg_s[s];
            p.pressure_raw[e] = (float)lg_s[e];
            p.pressure_rel[e] = tot > 0.0 ? (float)(lg_s[e] * p.S / tot) : 1.0f;
        }
        if (e == 0) {
            *p.step_counter = step + 1;
            *p.done_counter = 0u;
        }
    }
}

}  // namespace gimbal
