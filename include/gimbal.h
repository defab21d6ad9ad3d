/*
 * gimbal.h -- C ABI of libgimbal: the data-parallel hot path behind Gimbal's coordinated
 * MoE scheduling (arxiv/paper_2606_15177), hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * Citations are PAPER.md:<line> (+ section / equation) and DESIGN.md "R<n>" for the
 * readings taken where the paper is silent.
 *
 * Conventions (all entry points):
 *   - plain C, no C++ / torch types.  `gimbal_stream_t` is a cudaStream_t passed as void*.
 *   - every array argument is a DEVICE pointer owned by the caller unless the name ends in
 *     `_host` (the *_host entry points take HOST pointers, pinned for full speed, and do
 *     their own host<->device copies on the stream).  The library never frees or keeps a
 *     caller pointer past the call; scratch memory is a caller-owned device workspace whose
 *     size comes from the matching gimbal_*_workspace_bytes().
 *   - calls are asynchronous on `stream`, allocate nothing, never synchronise the host (the
 *     *_host variants synchronise the stream once, before returning), and can be captured
 *     in a CUDA graph.
 *   - return value: GIMBAL_OK or a negative error.  Host-detectable problems (NULL, shape,
 *     alignment, unsupported size) are reported here and nothing is launched.  Data errors
 *     only visible on the device (expert id out of range, invalid candidate) never trap:
 *     the affected outputs are NaN and bit 0 of the optional `status` word is set.
 *   - there is no CPU fallback: without a CUDA device of compute capability 10.x every
 *     compute entry point returns GIMBAL_ERR_UNSUPPORTED.
 */
#ifndef GIMBAL_H
#define GIMBAL_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define GIMBAL_API __attribute__((visibility("default")))
#else
#define GIMBAL_API
#endif

/* Version of this interface = the value gimbal_version() returns.  It changes whenever a struct layout, a buffer size or
 * an argument list of this header changes, so that a caller compiled against another header is refused instead of
 * reading or writing past its buffers:
 *   100  round 1
 *   300  gimbal_stats_state: step_counter is i64[2] (was [1]) and `reserved` became `abi_version`; gimbal_placement_cfg
 *        gained `encoding` and `flags`; gimbal_route_stats_host gained the leading `ctx`; gimbal_route_stats_static added.
 * Every gimbal_stats_state must carry abi_version = GIMBAL_ABI_VERSION (GIMBAL_ERR_INVALID_ARG otherwise, nothing is
 * launched); a caller can also compare gimbal_version() with the GIMBAL_ABI_VERSION it was compiled with at load time.   */
#define GIMBAL_ABI_VERSION 300

#define GIMBAL_OK 0
#define GIMBAL_ERR_INVALID_ARG (-1)
#define GIMBAL_ERR_UNSUPPORTED (-2)
#define GIMBAL_ERR_CUDA (-3)
#define GIMBAL_ERR_WORKSPACE (-4)

#define GIMBAL_SCORE_SOFTMAX 0
#define GIMBAL_SCORE_SIGMOID 1

#define GIMBAL_LOGITS_NONE 0 /* logits never leave the chip */
#define GIMBAL_LOGITS_OUT 1  /* logits computed and written to `logits` */
#define GIMBAL_LOGITS_IN 2   /* router GEMM skipped; gating reads `logits` */

#define GIMBAL_MODE_WINDOW 0
#define GIMBAL_MODE_EMA 1

#define GIMBAL_COUNTS_I32 0
#define GIMBAL_COUNTS_F32 1

#define GIMBAL_MAX_TOPK 8
#define GIMBAL_MAX_SOURCES 64

typedef void *gimbal_stream_t; /* cudaStream_t */

/* Router / gating shape.  The paper only says "lightweight router to select top-k experts
 * for each token"; score function, group limit and tie-break are set by the
 * model-shaped configs (R1, R3, R4).  Total order everywhere: (key descending,
 * index ascending), -0 == +0, NaN logits count as -inf.
 *   softmax : key_e = logit_e;  p = softmax over all E;  w_j = p_{id_j}
 *   sigmoid : s_e = sig32(logit_e);  key_e = fl32(s_e + select_bias_e);  w_j = s_{id_j}
 *   n_groups > 1 : E/n_groups contiguous experts per group; group score = fp32 sum (best
 *             first) of its group_score_topn largest keys; only the topk_groups best
 *             groups are eligible.
 *   renorm  : w_j /= sum of the k selected scores.   All weights are then * routed_scale.
 * Supported: E in {16,32,64,128,256}; 1 <= k <= 8; H % 64 == 0; S <= 64;
 *            n_groups | E with E/n_groups == 32 when n_groups > 1.                        */
typedef struct gimbal_router_cfg {
    int32_t L, H, E, k, S;
    int32_t score_fn, renorm, n_groups, topk_groups, group_score_topn;
    float routed_scale;
} gimbal_router_cfg;

/* Online routing profile (section 5.1).  All pointers are device memory.
 *   A_step [L,S,E] i32  out   this step's counts C (a3): tokens from DP source s routed to
 *                             expert e in layer l
 *   WINDOW mode: A_win += C; when (step+1) % window_len == 0 the window
 *     is published (A_pub = A_win, B_pub = B) and A_win is zeroed.
 *   A_win  [L,S,E] i32  inout   A_pub [L,S,E] i32 out   B_pub [L,E] i32 out
 *   EMA mode (BASELINE.json; R2): A_ema = fl32(ema_decay * A_ema + C), un-normalised.
 *   A_ema  [L,S,E] f32  inout
 *   B      [L,E]  i32 (WINDOW) / f32 (EMA)  out   B[l,e] = sum_s A[l,s,e] of the live profile
 *                             (A_win after this step's accumulation and before any reset,
 *                             or A_ema)
 *   pressure_raw [S] f32 out  MoE pressure of DP engine s: tokens processed by experts on its
 *                             EP ranks, sum_l sum_{g: dp_of_rank[g]=s} L[l,g]
 *   pressure_rel [S] f32 out  the same normalised to mean 1 (R14)
 *   step_counter [2] i64 inout  [0] device-side step index, incremented by every call that covers the last layer;
 *                               [1] scratch of the library (a layer counter): zero it once with [0], it is 0 between calls
 *   status [1] i32 inout|NULL  bit 0 set on device-side data errors                        */
typedef struct gimbal_stats_state {
    int32_t mode, window_len;
    float ema_decay;
    int32_t abi_version;   /* = GIMBAL_ABI_VERSION: the header this state was laid out by (step_counter [2]) */
    int32_t *A_step;
    int32_t *A_win;
    int32_t *A_pub;
    int32_t *B_pub;
    float *A_ema;
    void *B;
    float *pressure_raw;
    float *pressure_rel;
    int64_t *step_counter;
    int32_t *status;
} gimbal_stats_state;

/* Placement problem (section 5.2).  A placement is stored slot -> expert:
 * int16 [L,NS], NS = G*slots_per_rank, slot j of a layer lives on rank j / slots_per_rank.
 * x[l,e,g] in {0,1} = rank g hosts expert e.  With redundant slots (NS > E,
 * DESIGN.md R12) an expert may be hosted by r >= 1 ranks and its tokens split evenly over
 * them.  A valid placement hosts every expert at least once and never twice on one rank.
 * counts_dtype says whether A and B hold int32 or float.
 *   encoding  of the `candidates` of gimbal_eval_placements:
 *             SLOT_TO_EXPERT_I16  [P,L,NS] int16, as above (any supported shape);
 *             EXPERT_TO_RANK_U8   [P,L,E] uint8, byte e = the rank hosting expert e; only without
 *                                 replicas (NS == E) and E in {16,32,64,128,256}.  Half the bytes.
 *   flags     GIMBAL_PLACE_TRUSTED: the caller guarantees that every candidate is valid and hosts
 *             as many copies of each expert as x0 (true of anything made from x0 by slot exchanges,
 *             e.g. the output of gimbal_refine_placement or a rebalancer's own proposals); the
 *             validation pass is skipped.  A candidate that breaks the promise gets finite but
 *             meaningless numbers -- never a fault (ids are masked to the tables).
 * Supported: E <= 256 and even, G a power of two <= 64, slots_per_rank <= 16, G*slots_per_rank even, S <= 64.  An `encoding` other than the two
 * below or a bit of `flags` the library does not know is GIMBAL_ERR_INVALID_ARG (it is what a struct laid out by an older
 * header would carry there).                                                                 */
#define GIMBAL_ENC_SLOT_TO_EXPERT_I16 0
#define GIMBAL_ENC_EXPERT_TO_RANK_U8 1
#define GIMBAL_PLACE_TRUSTED 1

typedef struct gimbal_placement_cfg {
    int32_t L, E, G, slots_per_rank, S;
    float alpha, beta, gamma; /* J = alpha*C_comm + beta*C_load + gamma*C_mig; paper's
                                 calibrated (1.0, 0.0025, 1.0); R6 */
    int32_t counts_dtype;
    int32_t encoding;
    int32_t flags;
} gimbal_placement_cfg;

/* Expert mapping (NEXT-3; "fuse source counting with expert mapping"): the
 * logical expert ids chosen by the router become PHYSICAL slot ids under a placement, in the
 * same kernel that counts.  The slots hosting expert e, in ascending order, are s_0 < ... <
 * s_{r-1}; token t (its index in the step's token list) is sent to s_{t mod r} -- the even split
 * over replicas that the objective assumes (R12, R18); r = 1 in the paper.
 *   rep_off   [L, E+1] i32   expert e of layer l owns rep_slots[l, rep_off[l,e] .. rep_off[l,e+1])
 *   rep_slots [L, NS]  i16   slot ids grouped by expert, ascending inside a group
 *       (both are written by gimbal_build_expert_map from a slot -> expert placement)
 *   phys_ids  [n_layers, T, k] i32 out   slot id per (token, choice), in the order of topk_ids;
 *       rank = slot / slots_per_rank; -1 if the placement does not host that expert            */
typedef struct gimbal_expert_map {
    const int32_t *rep_off;
    const int16_t *rep_slots;
    int32_t *phys_ids;
    int32_t NS;
} gimbal_expert_map;

/* Library / device probe.  gimbal_version() returns the library's GIMBAL_ABI_VERSION and never touches CUDA. */
GIMBAL_API int gimbal_version(void);
/* Writes the last CUDA / validation error string (NUL-terminated, truncated to n). */
GIMBAL_API void gimbal_last_error(char *buf, size_t n);

/* ---------------------------------------------------------------------------------------
 * gimbal_route_stats -- steps a1..a5 for layers [layer0, layer0+n_layers) of one step:
 *   a1 logits[i,t,e] = sum_h hidden[i,t,h] * w_router[layer0+i,e,h]   (bf16 in, fp32 accumulate)
 *                      + src_logit_bias[layer0+i, src(t), e]           (optional; workload skew)
 *   a2 top-k gating (see gimbal_router_cfg)  ->  topk_ids, topk_w (both optional outputs)
 *   a3 A_step[l,s,e] = #{(t,j): src(t)=s, ids[l,t,j]=e}
 *   a4 window / EMA update, a5 B and MoE pressure (see gimbal_stats_state); a4-a5 cover all
 *      L layers of the state and run only when layer0 + n_layers == L (last slice of a step).
 * Arguments
 *   hidden        [n_layers,T,H] bf16, row-major, 16-byte aligned         (NULL if LOGITS_IN)
 *   w_router      [L,E,H] bf16 (row e = expert e's weights, K-major)      (NULL if LOGITS_IN)
 *   select_bias   [L,E] f32 | NULL     added to the sigmoid score for selection only
 *   src_logit_bias[L,S,E] f32 | NULL
 *   src_offsets   [S+1] i32            tokens are concatenated by source DP engine
 *                                      (PAPER.md:31); src_offsets[S] == T; empty sources ok
 *   logits        [n_layers,T,E] f32   written (OUT), read (IN) or ignored (NONE); holds the
 *                                      post-bias values fl32(acc + src_logit_bias)
 *   topk_ids      [n_layers,T,k] i32 | NULL   best first
 *   topk_w        [n_layers,T,k] f32 | NULL
 *   cur_placement [L,NS] i16 | NULL,  dp_of_rank [G] i32 | NULL : needed for the pressure
 *                                      outputs only (both NULL: pressure is left untouched)
 *   G, slots_per_rank                  shape of cur_placement
 *   map           | NULL               expert mapping: phys_ids written next to the counts
 * Stream order: the call behaves as if its kernels ran one after the other behind everything
 * enqueued on `stream` before it.  Internally the update kernel (a4-a5) and, when every layer of
 * the call is a single tile (T <= 256 and n_layers <= #SMs / 2), the router kernel are launched
 * with programmatic stream serialization: they may be SCHEDULED while the previous kernel on the
 * stream still runs and wait for it (griddepcontrol.wait) before their first global access.  In
 * that regime A_step is stored by one CTA pair per layer instead of accumulated, so it is never
 * zeroed first.  Capturable in a CUDA graph (programmatic edges).  See GIMBAL_OPT_PDL for the
 * opt-in that lets the router kernel overlap the previous step's update, and for plain launches.
 * Errors: INVALID_ARG (NULL / shape / alignment), UNSUPPORTED (shape outside the compiled
 * range, no sm_100 device), WORKSPACE (workspace_bytes too small), CUDA.                  */
GIMBAL_API size_t gimbal_route_stats_workspace_bytes(const gimbal_router_cfg *cfg, int n_layers, int T);

GIMBAL_API int gimbal_route_stats(const gimbal_router_cfg *cfg, int layer0, int n_layers, int T,
                       const void *hidden, const void *w_router,
                       const float *select_bias, const float *src_logit_bias,
                       const int32_t *src_offsets, int logits_mode, float *logits,
                       int32_t *topk_ids, float *topk_w,
                       const int16_t *cur_placement, const int32_t *dp_of_rank, int G, int slots_per_rank,
                       gimbal_stats_state *state, const gimbal_expert_map *map /* | NULL */,
                       void *workspace, size_t workspace_bytes, gimbal_stream_t stream);

/* ---------------------------------------------------------------------------------------
 * gimbal_route_stats_static -- gimbal_route_stats for callers that have no device memory to give.
 *
 * Who needs it.  gimbal_route_stats wants a caller-owned workspace (the per-layer pressure partials and the
 * layer counter of the a4-a5 update kernel).  A scheduler thread that lives inside a serving engine often
 * cannot provide one: the engine has already handed all free HBM to its KV-cache pool, so a cudaMalloc made
 * after start-up fails or steals from that pool; and a cudaMalloc / cudaFree issued from a side thread
 * synchronises the whole device and stalls the decode loop it sits next to.  For those callers the scratch
 * lives inside the library: a file-scope `static __device__` array of GIMBAL_STATIC_SCRATCH_BYTES (64 KiB)
 * that every GPU on which the library's code is loaded keeps until the process exits.
 *
 * Arguments, outputs, stream order and errors are those of gimbal_route_stats, minus `workspace` /
 * `workspace_bytes`; inputs, outputs and the state are still the caller's device memory.  Results are
 * bit-identical to gimbal_route_stats on the same inputs (same kernels, same launch configuration).
 *
 * Limit.  The shape must satisfy gimbal_route_stats_workspace_bytes(cfg, ..) <= GIMBAL_STATIC_SCRATCH_BYTES,
 * i.e. L * S <= 8128 (the DeepSeek-V3 shape has L * S = 928).  A larger shape is refused with
 * GIMBAL_ERR_WORKSPACE and a message that states both sizes; nothing is launched.
 *
 * Set-up.  The first call on each device (the device current at the call) resolves the array's device
 * address with cudaGetSymbolAddress -- the array's name in host code is only a handle, not something a
 * kernel can dereference -- and remembers it for that device.  That first call may make the runtime load
 * the library's device code, so make it once per device BEFORE any stream capture and before the part of
 * the program that must not stall.  If the look-up fails the call returns GIMBAL_ERR_CUDA.
 *
 * No allocation.  Neither the set-up nor any later call uses cudaMalloc, cudaFree, a memory pool or any
 * other allocating routine (host or device); with gimbal_kernel_timing switched on, the timing hooks'
 * events exist already.
 *
 * Sharing.  There is ONE array per device, shared by every call, every stream and every host thread of
 * the process, and it still holds whatever the previous call left there.  The entry point therefore
 * zeroes the part it is about to use whenever the shape's scratch layout differs from that of the previous
 * call on the device (the layer counter has to start at 0; the partials are always written before they
 * are read).  Two calls whose kernels can overlap on the GPU -- different streams, or the same step issued
 * from two threads -- race on the array and give wrong pressure values or a step that never completes its
 * update: serialise them (one stream, or events), or give the concurrent caller its own workspace through
 * gimbal_route_stats.                                                                              */
#define GIMBAL_STATIC_SCRATCH_BYTES 65536
GIMBAL_API int gimbal_route_stats_static(const gimbal_router_cfg *cfg, int layer0, int n_layers, int T,
                              const void *hidden, const void *w_router,
                              const float *select_bias, const float *src_logit_bias,
                              const int32_t *src_offsets, int logits_mode, float *logits,
                              int32_t *topk_ids, float *topk_w,
                              const int16_t *cur_placement, const int32_t *dp_of_rank, int G, int slots_per_rank,
                              gimbal_stats_state *state, const gimbal_expert_map *map /* | NULL */,
                              gimbal_stream_t stream);

/* Inverse of a slot -> expert placement [L,NS] for gimbal_expert_map: rep_off [L,E+1] and
 * rep_slots [L,NS] (device, caller-owned).  Ids out of range set bit 0 of `status`.         */
GIMBAL_API int gimbal_build_expert_map(int L, int E, int G, int slots_per_rank, const int16_t *placement,
                            int32_t *rep_off, int16_t *rep_slots, int32_t *status, gimbal_stream_t stream);

/* Context of the *_host entry points that overlap copies with kernels: a private copy stream and
 * its events on the device that is current at creation.  One context serves one host thread at a
 * time; create one per thread / device.  Creation allocates (the only entry point that does);
 * destroy waits for the copy stream.                                                          */
typedef struct gimbal_host_ctx gimbal_host_ctx;
GIMBAL_API int gimbal_host_ctx_create(gimbal_host_ctx **ctx);
GIMBAL_API int gimbal_host_ctx_destroy(gimbal_host_ctx *ctx);

/* Same step with the per-step inputs in HOST memory: hidden_host [n_layers,T,H] bf16 and
 * src_offsets_host [S+1] are copied to the device staging buffers the caller provides
 * (hidden_stage: at least 2 layers of [T,H] bf16; the copy of layer i+1 runs on ctx's stream while
 * layer i computes), and after the step A_step, B and both pressure vectors are copied back to
 * result_host (layout: A_step i32 [L,S,E] | B [L,E] | pressure_raw [S] | pressure_rel [S]),
 * gimbal_route_stats_result_bytes() bytes.  logits_mode is NONE.  Weights, biases, the
 * placement and the state stay device-resident (they persist across steps).  Synchronises
 * `stream` before returning.  INVALID_ARG if ctx is NULL or belongs to another device.        */
GIMBAL_API size_t gimbal_route_stats_result_bytes(const gimbal_router_cfg *cfg);
GIMBAL_API int gimbal_route_stats_host(gimbal_host_ctx *ctx, const gimbal_router_cfg *cfg, int T,
                            const void *hidden_host, const int32_t *src_offsets_host,
                            void *hidden_stage, size_t hidden_stage_bytes, int32_t *src_offsets_stage,
                            const void *w_router, const float *select_bias, const float *src_logit_bias,
                            const int16_t *cur_placement, const int32_t *dp_of_rank, int G, int slots_per_rank,
                            gimbal_stats_state *state, void *result_host,
                            void *workspace, size_t workspace_bytes, gimbal_stream_t stream);

/* ---------------------------------------------------------------------------------------
 * gimbal_eval_placements -- step a6: score P candidate placements against the profile.
 *   L[p,l,g] = sum_e B[l,e] x[l,e,g] / r[l,e]
 *   C_load   = sum_l sum_g (L[l,g] - mean_g L[l,g])^2
 *   C_comm   = sum_l sum_s sum_e sum_g A[l,s,e] D[s,g] x[l,e,g] / r[l,e]
 *   C_mig    = sum_l sum_e sum_g M[l,e,g] |x[l,e,g] - x0[l,e,g]|
 *   J        = alpha*C_comm + beta*C_load + gamma*C_mig
 *   maxload  = sum_l max_g L[l,g]                                           (R7)
 * r[l,e] is the CANDIDATE's replica count (R12): a candidate may replicate other experts
 * than x0 does.
 * Arguments
 *   candidates [P,L,NS] i16   slot -> expert (or [P,L,E] u8 expert -> rank, cfg->encoding); 16-byte aligned
 *   A [L,S,E], B [L,E]        i32 or f32 (cfg->counts_dtype), >= 0; B is an input of its own
 *                             because the paper collects it on another window (R9)
 *   D [S,G] f32 (>= 0)        source -> rank communication cost
 *   M [L,E,G] f32 (>= 0) | NULL   migration cost; NULL: M_scalar everywhere
 *   prev [L,NS] i16           x0, the placement before rebalancing (must be valid; an invalid x0
 *                             turns every output into NaN)
 *   out [P,5] f32             {J, C_load, C_comm, C_mig, maxload}; an invalid candidate (id or rank
 *                             out of range, an expert hosted nowhere, an expert twice on a rank, a
 *                             rank over capacity) gets five NaNs.  Validity is decided exactly: a
 *                             warp builds the candidate's x[e,g] bit matrix in shared memory and
 *                             reads every condition off it (skipped with GIMBAL_PLACE_TRUSTED).
 *                             C_mig adds up the entering and the leaving cells directly, so it is
 *                             exactly 0 for a candidate equal to x0.
 *   argmin [1] i32 | NULL     lowest index among the candidates of minimal J (NaNs skipped;
 *                             -1 if none is valid)
 * EXPERT_TO_RANK_U8 sums a rank's load with shared-memory float atomics: with f32 counts the last
 * bits of C_load depend on the order of the additions (integer counts below 2^24 are exact).    */
GIMBAL_API size_t gimbal_eval_placements_workspace_bytes(const gimbal_placement_cfg *cfg, int P);

GIMBAL_API int gimbal_eval_placements(const gimbal_placement_cfg *cfg, int P, const void *candidates,
                           const void *A, const void *B, const float *D, const float *M, float M_scalar,
                           const int16_t *prev, float *out, int32_t *argmin,
                           void *workspace, size_t workspace_bytes, gimbal_stream_t stream);

/* Candidates and results in HOST memory (cand_stage: device buffer of the candidates' size;
 * out_stage: device [P,5] f32).  Synchronises `stream` before returning.                  */
GIMBAL_API int gimbal_eval_placements_host(const gimbal_placement_cfg *cfg, int P, const void *candidates_host,
                                void *cand_stage, float *out_stage,
                                const void *A, const void *B, const float *D, const float *M, float M_scalar,
                                const int16_t *prev, float *out_host, int32_t *argmin_host,
                                void *workspace, size_t workspace_bytes, gimbal_stream_t stream);

/* ---------------------------------------------------------------------------------------
 * gimbal_eval_moves -- step a7: objective deltas of single moves from placement `cur`.
 * A move (l, slot_a, slot_b) exchanges the contents of two slots of layer l (a move into a
 * redundant slot is a swap with that slot).  delta equals J(moved) - J(cur) term by term:
 *   delta [n,5] f32 = {dJ, dC_load, dC_comm, dC_mig, dmaxload}
 * Same-rank moves and exchanges of two replicas of one expert give zeros; a move that would
 * put a second copy of an expert on a rank gives NaNs.
 *   moves [n,3] i32 | NULL   NULL = the whole neighbourhood in canonical order: for l in
 *                            [0,L), for a < b (a outer, b inner); then n_moves must equal
 *                            L*NS*(NS-1)/2
 *   best_per_layer [L] i32 | NULL  index (into the n moves) of the lowest dJ of each layer,
 *                            lowest index on ties, -1 if the layer has no valid move
 * Other arguments as in gimbal_eval_placements; `cur` and `prev` must be valid and host the same
 * number of copies of every expert (an exchange keeps them), else every delta is NaN.  The whole
 * neighbourhood runs in a kernel that stages the layer's per-slot rows in shared memory when they
 * fit (every BASELINE.json shape does), otherwise -- like an explicit list -- one thread per move.  */
GIMBAL_API size_t gimbal_eval_moves_workspace_bytes(const gimbal_placement_cfg *cfg);

GIMBAL_API int gimbal_eval_moves(const gimbal_placement_cfg *cfg, const int16_t *cur, const int16_t *prev,
                      int64_t n_moves, const int32_t *moves,
                      const void *A, const void *B, const float *D, const float *M, float M_scalar,
                      float *delta, int32_t *best_per_layer,
                      void *workspace, size_t workspace_bytes, gimbal_stream_t stream);

/* The per-call inputs in HOST memory: cur_host / prev_host [L,NS] and the optional move list
 * moves_host [n,3] are copied to their *_stage device buffers; best_host [L] (optional) and, when
 * delta_host is not NULL, delta [n,5] are copied back (delta_stage [n,5] always receives the
 * deltas on the device: a whole neighbourhood is 20 bytes per move, so a caller that only wants
 * the best move per layer leaves delta_host NULL).  Synchronises `stream` before returning.     */
GIMBAL_API int gimbal_eval_moves_host(const gimbal_placement_cfg *cfg, const int16_t *cur_host, const int16_t *prev_host,
                           int16_t *cur_stage, int16_t *prev_stage, int64_t n_moves, const int32_t *moves_host,
                           int32_t *moves_stage, const void *A, const void *B, const float *D, const float *M,
                           float M_scalar, float *delta_stage, float *delta_host /* | NULL */,
                           int32_t *best_stage, int32_t *best_host /* | NULL */,
                           void *workspace, size_t workspace_bytes, gimbal_stream_t stream);

/* ---------------------------------------------------------------------------------------
 * gimbal_greedy_place -- the online greedy placement heuristic (section
 * 5.3; R17), every layer in parallel.  Items are the slot contents of x0 (`prev`);
 * they are taken in order of hotness (B[l,e] + sum_s A[l,s,e]) / r (descending; expert index,
 * then slot index break ties) and each goes to the feasible rank (free slot, not already
 * holding that expert) with the lowest local score
 *     S[l,e,g] = alpha * sum_s A[l,s,e] D[s,g] / r  +  beta * (load placed on g so far + B[l,e]/r)
 *              + gamma * (M[l,e,g] if x0 does not host e on g, else 0)
 * ties: a placement that avoids migration first, then the less-filled rank,
 * then the lower rank index.  Scores are evaluated in IEEE double, one rounding per operation,
 * so the resulting placement is a pure function of the inputs (bit-exact against the oracle).
 *   out [L,NS] i16   slot -> expert; slot g*slots_per_rank + i = the i-th item given to rank g.
 *                    A layer whose x0 is invalid, or where an item finds no feasible rank, is
 *                    filled with -1 and bit 1 of `status` is set.
 *   status [1] i32 inout | NULL
 * Other arguments as in gimbal_eval_placements.  Needs no workspace.                       */
GIMBAL_API int gimbal_greedy_place(const gimbal_placement_cfg *cfg, const void *A, const void *B, const float *D,
                        const float *M, float M_scalar, const int16_t *prev, int16_t *out, int32_t *status,
                        gimbal_stream_t stream);

/* ---------------------------------------------------------------------------------------
 * gimbal_select_engines -- Algorithm 1, Global DP Engine Scheduling (section
 * 4.3; readings DESIGN.md R19), batched: B independent scheduler instances, each with N DP
 * engines and R incoming requests handled in order.  Per request: incomplete traces -> ordered
 * dispatch Next(E); else the KV rule (max kv > high_kv and max - min kv > large_gap -> the engine
 * with the lowest kv); else score_i = pre_rem_i + wait_i + comp_i + lambda_kv*kv_i +
 * lambda_moe*moe_i, ordered dispatch when max - min score < close_frac * len(r), otherwise the
 * argmin of (score, kv, i).  After each assignment comp[e*] += len(r).
 *   trace    [B,N,4] f32   {kv in [0,1], pre_rem tokens, wait tokens, moe = relative MoE pressure
 *                          (pressure_rel of gimbal_route_stats, mean 1)}; 16-byte aligned
 *   complete [B] u8 | NULL  0: this instance's traces are incomplete
 *   req_len  [B,R] f32      prefill tokens of the incoming requests
 *   comp     [B,N] f64 inout  compensation load; the caller zeroes it when it loads a fresh trace
 *   rr       [B] i32 inout    ordered-dispatch pointer
 *   engine   [B,R] i32 out    selected engine per request
 * Supported: 1 <= N <= 64.  Decisions are taken in IEEE double (bit-exact against the oracle). */
typedef struct gimbal_sched_cfg {
    int32_t N, R;
    float high_kv, large_gap;       /* 0.90, 0.10 */
    float lambda_kv, lambda_moe;    /* token-equivalent weights of P_kv, P_moe (R19) */
    float close_frac;               /* CLOSE threshold as a fraction of the request length (R19) */
} gimbal_sched_cfg;

GIMBAL_API int gimbal_select_engines(const gimbal_sched_cfg *cfg, int B, const float *trace, const uint8_t *complete,
                          const float *req_len, double *comp, int32_t *rr, int32_t *engine, gimbal_stream_t stream);

/* ---------------------------------------------------------------------------------------
 * gimbal_order_queues -- Algorithm 2, Request Scheduler with SJF and Aging (PAPER.md:179-200,
 * section 4.4; R20), batched over B waiting queues.  A request that has waited
 * now - arrival >= theta_age (5 s in the paper) is high priority; the others are
 * ordered by prefill length.  Total order: aged first, oldest first; then shortest prefill,
 * equal lengths oldest first; then the position in the input queue.
 *   arrival [B,Q] f32 seconds, prefill [B,Q] i32 tokens, qlen [B] i32 (requests in each queue, <= Q)
 *   order   [B,Q] i32 out: order[b,i] = input position of the i-th request to run; -1 past qlen[b]
 * Supported: Q <= 2048.                                                                     */
GIMBAL_API int gimbal_order_queues(int B, int Q, const float *arrival, const int32_t *prefill, const int32_t *qlen,
                        float now, float theta_age, int32_t *order, gimbal_stream_t stream);

/* ---------------------------------------------------------------------------------------
 * gimbal_refine_placement -- swap-based local search on top of gimbal_eval_moves (SURVEY.md
 * section 8f, NEXT-1; not in the paper, R21): `iters` rounds; in each round every layer
 * applies its best single slot exchange of the whole neighbourhood when
 *     dJ < -1e-4 * (alpha*|dC_comm| + beta*|dC_load| + gamma*|dC_mig|)
 * (a margin above fp32 rounding, so that the search cannot cycle on noise).  Asynchronous, no host
 * round trip between rounds.
 *   cur     [L,NS] i16 inout   placement being refined (must stay valid: x0's expert copies)
 *   delta   [L*NS*(NS-1)/2, 5] f32  scratch = the deltas of the last round (as gimbal_eval_moves)
 *   best    [L] i32            scratch = best move of each layer in the last round
 *   applied [L] i32 out | NULL number of exchanges applied per layer (zeroed by the call)
 * Other arguments as in gimbal_eval_moves (same workspace size).                            */
GIMBAL_API int gimbal_refine_placement(const gimbal_placement_cfg *cfg, int16_t *cur, const int16_t *prev, int iters,
                            const void *A, const void *B, const float *D, const float *M, float M_scalar,
                            float *delta, int32_t *best, int32_t *applied,
                            void *workspace, size_t workspace_bytes, gimbal_stream_t stream);

/* Process-wide switches for tests and A/B measurements (not for concurrent use; production keeps
 * the defaults).  They replace environment variables: nothing in the library reads the environment.
 *   GIMBAL_OPT_CTA_GROUP         0 (default: cta_group::2 when T > 128), 1 or 2: router GEMM pairing
 *   GIMBAL_OPT_FUSE_GATE         1 (default): gating + histogram in the GEMM epilogue; 0: GEMM writes
 *                                logits, the standalone gating kernel reads them (needs LOGITS_OUT)
 *   GIMBAL_OPT_SCORE_GENERIC     0 (default); 1: the shape-generic scoring kernel even where a
 *                                specialised one exists
 *   GIMBAL_OPT_CHECK_SCORES_ALL  0 (default); 1: place_check_kernel scores every valid candidate with
 *                                the candidate's own replica counts (the path otherwise taken only by
 *                                candidates whose replica counts differ from x0's)
 *   GIMBAL_OPT_HIST_AGG          1 (default): the router GEMM epilogue counts a warp's 32 tokens by columns
 *                                (bit-matrix transpose, one shared atomic per lane and 32 experts) when they
 *                                share one source; 0: one predicated shared atomic per selected logit
 *   GIMBAL_OPT_SCORE_TMA         1 (default): on the 9-slots x 32-ranks x 256-experts shape with a scalar M, the
 *                                scoring-only pass (GIMBAL_PLACE_TRUSTED) receives its candidate rows by TMA;
 *                                0: per-lane global loads as on every other shape
 *   GIMBAL_OPT_EPI_PARTS         0 (default: auto), 1 or 2: epilogue warps per TMEM lane quadrant of the fused router kernel.
 *                                2 (E >= 128, counts only) splits a row's experts between two warps that meet in shared
 *                                memory; auto picks it when no CTA pair gets more than two tiles (small-batch regime, where
 *                                the epilogue is not hidden behind the MMAs)
 *   GIMBAL_OPT_PDL               1 (default): stats_update_kernel, and the fused router kernel in the one-tile-per-layer regime,
 *                                are launched with programmatic stream serialization and wait for their predecessor themselves
 *                                before their first global access (launch latency and prologues overlap; always safe);
 *                                2: the caller PROMISES that the inputs of gimbal_route_stats (hidden, w_router, biases,
 *                                src_offsets) were complete before the operation that precedes the call on the stream was
 *                                enqueued -- e.g. steps replayed from pre-staged buffers -- and the router kernel then waits
 *                                only before it stores its counts: it overlaps the previous step's update entirely;
 *                                0: plain launches
 *   GIMBAL_OPT_FUSE_UPDATE       1 (default): a whole-step call (layer0 = 0, n_layers = L) in the one-tile-per-layer regime runs
 *                                a4-a5 inside the router kernel (the CTA pair that stored a layer's counts updates that layer, the
 *                                last pair finishes the step): one kernel per step; 0: separate stats_update_kernel          */
#define GIMBAL_OPT_CTA_GROUP 0
#define GIMBAL_OPT_FUSE_GATE 1
#define GIMBAL_OPT_SCORE_GENERIC 2
#define GIMBAL_OPT_CHECK_SCORES_ALL 3
#define GIMBAL_OPT_HIST_AGG 4
#define GIMBAL_OPT_SCORE_TMA 5
#define GIMBAL_OPT_EPI_PARTS 6
#define GIMBAL_OPT_PDL 7
#define GIMBAL_OPT_FUSE_UPDATE 8
#define GIMBAL_OPT_COUNT_ 9
GIMBAL_API int gimbal_set_option(int option, int value);
GIMBAL_API int gimbal_get_option(int option, int *value);

/* Counters for bench.py: kernels launched by this library since load. */
GIMBAL_API int64_t gimbal_launch_count(void);

/* Measurement hooks for bench.py.  With timing enabled the library records a pair of CUDA
 * events on the caller's stream around each launch of its four main kernels (never enable
 * this while capturing a CUDA graph).  gimbal_kernel_elapsed_ms() waits for the most recent
 * launch of kernel `which` to finish and returns its device time in milliseconds.           */
#define GIMBAL_KERNEL_ROUTER 0 /* router GEMM (+ fused gating / histogram)  a1-a3 */
#define GIMBAL_KERNEL_GATE 1   /* standalone gating + histogram              a2-a3 */
#define GIMBAL_KERNEL_SCORE 2  /* placement scoring                          a6    */
#define GIMBAL_KERNEL_MOVES 3  /* move deltas                                a7    */
#define GIMBAL_KERNEL_GREEDY 4 /* greedy placement heuristic                 NEXT-1 */
#define GIMBAL_KERNEL_CHECK 5  /* exact candidate validation                 a6    */
GIMBAL_API int gimbal_kernel_timing(int enable);
GIMBAL_API int gimbal_kernel_elapsed_ms(int which, float *ms);

#ifdef __cplusplus
}
#endif
#endif /* GIMBAL_H */
