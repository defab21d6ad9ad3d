/*
 * gimbal_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU statement of what the Gimbal hot path computes
 * (arxiv/paper_2606_15177; citations are PAPER.md:<line> plus section / equation, and
 * DESIGN.md "R<n>" for the readings taken where the paper is silent).  fp64 / int64
 * throughout unless a decision precision is fixed (see oracle_gate, tier 1).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may call this file.  It shares no code, header, table or constant generator with the
 * CUDA path under paper_2606_15177_b200/csrc, and neither includes the other.
 *
 * There is no blocking, fusion or re-ordering here beyond what the definitions state;
 * OpenMP (when enabled) only splits independent tokens / candidates / moves.
 *
 * Parity pins (tests/test_oracle_pins.py): every function below is pinned against
 * something other than itself -- hand-computed worked examples (tests/golden/), closed
 * forms, invariants, numpy library routines, brute-force enumeration.  Numeric parity
 * with values PRINTED BY THE PAPER is unpinned: the paper prints none for this path
 * (Table 1, holds raw counts only).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_SOFTMAX 0
#define ORACLE_SIGMOID 1

/* ------------------------------------------------------------------------------------ */
/* a1  Router logits.  logits[t,e] = sum_h hidden[t,h] * W[e,h]  ("lightweight
 *     router"; BASELINE.json north_star: "router GEMM (hidden x W_router)", oracle "in fp64
 *     from the same bf16 inputs").  Every bf16*bf16 product is exact in fp64.
 *     + src_logit_bias[src(t), e] (benchmark scaffolding, R5/section 4).          */
/* ------------------------------------------------------------------------------------ */
static double bf16_to_double(uint16_t b)
{
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

static int source_of_token(const int32_t *src_offsets, int S, int t)
{
    /* tokens of a step are concatenated by source; empty sources allowed */
    for (int s = 0; s < S; ++s)
        if (t >= src_offsets[s] && t < src_offsets[s + 1]) return s;
    return -1;
}

void oracle_router_logits(const uint16_t *hidden /*[T,H] bf16 bits*/,
                          const uint16_t *w /*[E,H] bf16 bits*/,
                          const float *src_logit_bias /*[S,E] or NULL*/,
                          const int32_t *src_offsets /*[S+1]*/,
                          int T, int H, int E, int S,
                          double *logits64 /*[T,E]*/, float *logits32 /*[T,E]*/)
{
#pragma omp parallel for schedule(static)
    for (int t = 0; t < T; ++t) {
        int s = source_of_token(src_offsets, S, t);
        for (int e = 0; e < E; ++e) {
            double acc = 0.0;
            for (int h = 0; h < H; ++h)
                acc += bf16_to_double(hidden[(size_t)t * H + h]) * bf16_to_double(w[(size_t)e * H + h]);
            if (src_logit_bias && s >= 0) acc += (double)src_logit_bias[(size_t)s * E + e];
            logits64[(size_t)t * E + e] = acc;
            logits32[(size_t)t * E + e] = (float)acc;
        }
    }
}

/* ------------------------------------------------------------------------------------ */
/* a2  Gating.  The paper only says "select top-k experts for each token";
 *     the score function, group limit and tie-break are BASELINE.json's (R1,
 *     R3, R4).  Total order everywhere: (key descending, index ascending); -0 == +0; a NaN
 *     logit is treated as -inf.
 *
 *     tier 0: the plain definition, keys in fp64.
 *     tier 1: the DECISION PRECISION of the contract -- keys in fp32, sigmoid through the
 *             specified routine sig32 (DESIGN.md section 5 states it operation by
 *             operation; this is an independent restatement of that text).  Softmax mode
 *             selects on the raw fp32 logits, so both tiers coincide there.
 *     Weights are always the plain definition in fp64 from the fp32 logits.              */
/* ------------------------------------------------------------------------------------ */
float oracle_sig32(float x)
{
    /* every step is one correctly-rounded IEEE-754 binary32 op.
       Compile with -ffp-contract=off. */
    const float LOG2E = 0x1.715476p+0f;
    const float MAGIC = 12582912.0f; /* 1.5 * 2^23 */
    float t = -x * LOG2E;
    t = fminf(fmaxf(t, -125.0f), 125.0f);
    float r = t + MAGIC;
    float n = r - MAGIC;
    float f = t - n;
    float p = 0x1.444p-13f;
    p = fmaf(p, f, 0x1.5f48cp-10f);
    p = fmaf(p, f, 0x1.3b2a1cp-7f);
    p = fmaf(p, f, 0x1.c6aeccp-5f);
    p = fmaf(p, f, 0x1.ebfbep-3f);
    p = fmaf(p, f, 0x1.62e43p-1f);
    p = fmaf(p, f, 1.0f);
    uint32_t pb, rb;
    memcpy(&pb, &p, 4);
    memcpy(&rb, &r, 4);
    uint32_t eb = pb + (rb << 23); /* p * 2^n */
    float e;
    memcpy(&e, &eb, 4);
    float d = 1.0f + e;
    return 1.0f / d;
}

void oracle_sig32_array(const float *x, int n, float *out)
{
    for (int i = 0; i < n; ++i) out[i] = oracle_sig32(x[i]);
}

typedef struct {
    int32_t E, k, score_fn, renorm, n_groups, topk_groups, group_score_topn;
    double routed_scale;
} oracle_gate_cfg;

/* a > b under (key desc, index asc): does (ka, ia) come before (kb, ib)? */
static int before(double ka, int ia, double kb, int ib)
{
    if (ka > kb) return 1;
    if (ka < kb) return 0;
    return ia < ib;
}

static void gate_row(const oracle_gate_cfg *c, const float *x32, const float *select_bias, int tier,
                     int32_t *ids, double *wts)
{
    const int E = c->E, k = c->k;
    double *x = (double *)malloc(sizeof(double) * E);    /* sanitised logits */
    double *key = (double *)malloc(sizeof(double) * E);
    double *sc = (double *)malloc(sizeof(double) * E);   /* unbiased scores (weights) */
    char *elig = (char *)malloc(E);
    char *taken = (char *)calloc(E, 1);

    for (int e = 0; e < E; ++e) {
        float v = x32[e];
        if (v != v) v = -INFINITY;
        x[e] = (double)v;
    }
    if (c->score_fn == ORACLE_SOFTMAX) {
        /* selection key = the logit itself (softmax is monotone) */
        double mx = -INFINITY, sum = 0.0;
        for (int e = 0; e < E; ++e) if (x[e] > mx) mx = x[e];
        for (int e = 0; e < E; ++e) { sc[e] = (mx == -INFINITY) ? 1.0 : exp(x[e] - mx); sum += sc[e]; }
        for (int e = 0; e < E; ++e) { sc[e] /= sum; key[e] = x[e]; }
    } else {
        for (int e = 0; e < E; ++e) {
            double b = select_bias ? (double)select_bias[e] : 0.0;
            sc[e] = 1.0 / (1.0 + exp(-x[e]));
            if (tier == 0) key[e] = sc[e] + b;
            else {
                float s32 = oracle_sig32((float)x[e]);
                float k32 = select_bias ? (s32 + select_bias[e]) : s32;
                key[e] = (double)k32;
            }
        }
    }
    for (int e = 0; e < E; ++e) { if (key[e] != key[e]) key[e] = -INFINITY; elig[e] = 1; }

    if (c->n_groups > 1) {
        /* group-limited routing (R1): contiguous groups of E/n_groups experts;
           group score = sum of its group_score_topn largest keys (added best first, in
           the tier's precision); keep the topk_groups best groups. */
        const int ng = c->n_groups, gs = E / ng;
        double *gscore = (double *)malloc(sizeof(double) * ng);
        char *gkeep = (char *)calloc(ng, 1);
        for (int q = 0; q < ng; ++q) {
            char *used = (char *)calloc(gs, 1);
            double acc = 0.0; float acc32 = 0.0f;
            for (int j = 0; j < c->group_score_topn; ++j) {
                int best = -1;
                for (int i = 0; i < gs; ++i)
                    if (!used[i] && (best < 0 || before(key[q * gs + i], i, key[q * gs + best], best))) best = i;
                used[best] = 1;
                if (j == 0) { acc = key[q * gs + best]; acc32 = (float)key[q * gs + best]; }
                else { acc += key[q * gs + best]; acc32 = acc32 + (float)key[q * gs + best]; }
            }
            gscore[q] = (tier == 0) ? acc : (double)acc32;
            if (gscore[q] != gscore[q]) gscore[q] = -INFINITY;
            free(used);
        }
        for (int j = 0; j < c->topk_groups; ++j) {
            int best = -1;
            for (int q = 0; q < ng; ++q)
                if (!gkeep[q] && (best < 0 || before(gscore[q], q, gscore[best], best))) best = q;
            gkeep[best] = 1;
        }
        for (int e = 0; e < E; ++e) elig[e] = gkeep[e / gs];
        free(gscore); free(gkeep);
    }

    /* top-k of the eligible keys, best first */
    double selsum = 0.0;
    for (int j = 0; j < k; ++j) {
        int best = -1;
        for (int e = 0; e < E; ++e)
            if (elig[e] && !taken[e] && (best < 0 || before(key[e], e, key[best], best))) best = e;
        taken[best] = 1;
        ids[j] = best;
        selsum += sc[best];
    }
    for (int j = 0; j < k; ++j) {
        double wj = sc[ids[j]];
        if (c->renorm) wj /= selsum;
        wts[j] = wj * c->routed_scale;
    }
    free(x); free(key); free(sc); free(elig); free(taken);
}

void oracle_gate(const oracle_gate_cfg *c, const float *logits32 /*[T,E]*/, const float *select_bias /*[E]|NULL*/,
                 int T, int tier, int32_t *ids /*[T,k]*/, double *wts /*[T,k]*/)
{
#pragma omp parallel for schedule(static)
    for (int t = 0; t < T; ++t)
        gate_row(c, logits32 + (size_t)t * c->E, select_bias, tier, ids + (size_t)t * c->k, wts + (size_t)t * c->k);
}

/* ------------------------------------------------------------------------------------ */
/* a3  Source x expert counts: C[s,e] = #{(t,j): src(t)=s and ids[t,j]=e}
 *     ("A_{l,s,e} is the number of tokens from DP source s that are routed to expert e in
 *     layer l", section 5.1).                                               */
/* ------------------------------------------------------------------------------------ */
void oracle_counts(const int32_t *ids /*[T,k]*/, const int32_t *src_offsets /*[S+1]*/,
                   int T, int k, int S, int E, int64_t *C /*[S,E]*/)
{
    memset(C, 0, sizeof(int64_t) * (size_t)S * E);
    for (int t = 0; t < T; ++t) {
        int s = source_of_token(src_offsets, S, t);
        if (s < 0) continue;
        for (int j = 0; j < k; ++j) C[(size_t)s * E + ids[(size_t)t * k + j]] += 1;
    }
}

/* ------------------------------------------------------------------------------------ */
/* a4  Window / EMA update of the profile (n = L*S*E elements).
 *     WINDOW: counts accumulate over a profiling window and are published at its end
 *     ("during a profiling window", "At the end of each
 *     profiling window, Gimbal aggregates ...").  EMA (BASELINE.json; R2):
 *     un-normalised A <- d*A + C.                                                        */
/* ------------------------------------------------------------------------------------ */
void oracle_update_window(int64_t *A_win, const int64_t *C, int64_t *A_pub, int64_t n,
                          int64_t step, int64_t window_len, int32_t *published)
{
    for (int64_t i = 0; i < n; ++i) A_win[i] += C[i];
    *published = ((step + 1) % window_len) == 0;
    if (*published) {
        for (int64_t i = 0; i < n; ++i) { A_pub[i] = A_win[i]; A_win[i] = 0; }
    }
}

void oracle_update_ema(double *A_ema, const int64_t *C, int64_t n, double decay)
{
    for (int64_t i = 0; i < n; ++i) A_ema[i] = decay * A_ema[i] + (double)C[i];
}

/* ------------------------------------------------------------------------------------ */
/* placements.  A placement is stored slot -> expert: slot j of layer l lives on rank
 * j / slots_per_rank.  x[l,e,g] in {0,1} says rank g hosts expert e; with
 * redundant slots (R12) an expert may be hosted by r_{l,e} = sum_g x >= 1 ranks
 * and its tokens split evenly over them.  Valid: ids in range, every expert hosted at
 * least once, never twice on one rank.                                                   */
/* ------------------------------------------------------------------------------------ */
static int build_x(const int16_t *place /*[NS]*/, int E, int G, int sp, double *x /*[E,G]*/, double *r /*[E]*/)
{
    memset(x, 0, sizeof(double) * (size_t)E * G);
    for (int j = 0; j < G * sp; ++j) {
        int e = place[j], g = j / sp;
        if (e < 0 || e >= E) return 0;
        if (x[(size_t)e * G + g] != 0.0) return 0;
        x[(size_t)e * G + g] = 1.0;
    }
    for (int e = 0; e < E; ++e) {
        r[e] = 0.0;
        for (int g = 0; g < G; ++g) r[e] += x[(size_t)e * G + g];
        if (r[e] < 1.0) return 0;
    }
    return 1;
}

/* a5  B[l,e] = sum_s A[l,s,e]; L[l,g] = sum_e B[l,e] x[l,e,g] / r_{l,e}
 *     (r=1 in the paper); MoE pressure of DP engine s = tokens processed
 *     by experts on its associated EP ranks, raw and normalised to mean 1
 *     ("normalized ... relative penalty"; R14).                    */
int oracle_derived(const double *A /*[L,S,E]*/, const int16_t *place /*[L,NS]*/, const int32_t *dp_of_rank /*[G]*/,
                   int L, int S, int E, int G, int sp,
                   double *B /*[L,E]*/, double *Lrank /*[L,G]*/, double *pressure_raw /*[S]*/, double *pressure_rel /*[S]*/)
{
    double *x = (double *)malloc(sizeof(double) * (size_t)E * G), *r = (double *)malloc(sizeof(double) * E);
    int ok = 1;
    for (int s = 0; s < S; ++s) pressure_raw[s] = 0.0;
    for (int l = 0; l < L; ++l) {
        for (int e = 0; e < E; ++e) {
            double b = 0.0;
            for (int s = 0; s < S; ++s) b += A[((size_t)l * S + s) * E + e];
            B[(size_t)l * E + e] = b;
        }
        if (!build_x(place + (size_t)l * G * sp, E, G, sp, x, r)) { ok = 0; break; }
        for (int g = 0; g < G; ++g) {
            double lg = 0.0;
            for (int e = 0; e < E; ++e) lg += B[(size_t)l * E + e] * x[(size_t)e * G + g] / r[e];
            Lrank[(size_t)l * G + g] = lg;
            pressure_raw[dp_of_rank[g]] += lg;
        }
    }
    double tot = 0.0;
    for (int s = 0; s < S; ++s) tot += pressure_raw[s];
    for (int s = 0; s < S; ++s) pressure_rel[s] = tot > 0.0 ? pressure_raw[s] * S / tot : 1.0;
    free(x); free(r);
    return ok;
}

/* a6  Placement objective, evaluated literally as printed (section 5.2):
 *       L[l,g]  = sum_e B[l,e] x[l,e,g] / r[l,e]
 *       C_load  = sum_l sum_g (L[l,g] - Lbar_l)^2
 *       C_comm  = sum_l sum_s sum_e sum_g A[l,s,e] D[s,g] x[l,e,g]/r
 *       C_mig   = sum_l sum_e sum_g M[l,e,g] |x[l,e,g] - x0[l,e,g]|
 *       J       = alpha C_comm + beta C_load + gamma C_mig     (R6)
 *       maxload = sum_l max_g L[l,g]                           (BASELINE.json; R7)
 *     out[5] = {J, C_load, C_comm, C_mig, maxload}; per-layer terms optionally in
 *     per_layer[L,4] = {C_load_l, C_comm_l, C_mig_l, maxload_l}.  Returns 0 and fills NaN
 *     if the candidate (or x0) is invalid.                                               */
int oracle_objective(const int16_t *cand /*[L,NS]*/, const int16_t *prev /*[L,NS]*/,
                     const double *A /*[L,S,E]*/, const double *B /*[L,E]*/, const double *D /*[S,G]*/,
                     const double *M /*[L,E,G] or NULL*/, double M_scalar,
                     int L, int S, int E, int G, int sp, double alpha, double beta, double gamma,
                     double *out /*[5]*/, double *per_layer /*[L,4] or NULL*/)
{
    const int NS = G * sp;
    double *x = (double *)malloc(sizeof(double) * (size_t)E * G), *r = (double *)malloc(sizeof(double) * E);
    double *x0 = (double *)malloc(sizeof(double) * (size_t)E * G), *r0 = (double *)malloc(sizeof(double) * E);
    double c_load = 0.0, c_comm = 0.0, c_mig = 0.0, maxload = 0.0;
    int ok = 1;
    for (int l = 0; l < L && ok; ++l) {
        if (!build_x(cand + (size_t)l * NS, E, G, sp, x, r) || !build_x(prev + (size_t)l * NS, E, G, sp, x0, r0)) { ok = 0; break; }
        const double *Al = A + (size_t)l * S * E, *Bl = B + (size_t)l * E;
        double load_l = 0.0, comm_l = 0.0, mig_l = 0.0, max_l = -INFINITY, mean = 0.0;
        double *Lg = (double *)malloc(sizeof(double) * G);
        for (int g = 0; g < G; ++g) {
            Lg[g] = 0.0;
            for (int e = 0; e < E; ++e) Lg[g] += Bl[e] * x[(size_t)e * G + g] / r[e];
            mean += Lg[g];
        }
        mean /= G;
        for (int g = 0; g < G; ++g) {
            load_l += (Lg[g] - mean) * (Lg[g] - mean);
            if (Lg[g] > max_l) max_l = Lg[g];
        }
        for (int s = 0; s < S; ++s)
            for (int e = 0; e < E; ++e)
                for (int g = 0; g < G; ++g)
                    comm_l += Al[(size_t)s * E + e] * D[(size_t)s * G + g] * x[(size_t)e * G + g] / r[e];
        for (int e = 0; e < E; ++e)
            for (int g = 0; g < G; ++g) {
                double m = M ? M[((size_t)l * E + e) * G + g] : M_scalar;
                mig_l += m * fabs(x[(size_t)e * G + g] - x0[(size_t)e * G + g]);
            }
        free(Lg);
        c_load += load_l; c_comm += comm_l; c_mig += mig_l; maxload += max_l;
        if (per_layer) { per_layer[l * 4 + 0] = load_l; per_layer[l * 4 + 1] = comm_l; per_layer[l * 4 + 2] = mig_l; per_layer[l * 4 + 3] = max_l; }
    }
    if (ok) {
        out[0] = alpha * c_comm + beta * c_load + gamma * c_mig;
        out[1] = c_load; out[2] = c_comm; out[3] = c_mig; out[4] = maxload;
    } else {
        for (int i = 0; i < 5; ++i) out[i] = NAN;
    }
    free(x); free(r); free(x0); free(r0);
    return ok;
}

void oracle_objective_batch(const int16_t *cands /*[P,L,NS]*/, int P, const int16_t *prev,
                            const double *A, const double *B, const double *D, const double *M, double M_scalar,
                            int L, int S, int E, int G, int sp, double alpha, double beta, double gamma,
                            double *out /*[P,5]*/)
{
#pragma omp parallel for schedule(dynamic, 4)
    for (int p = 0; p < P; ++p)
        oracle_objective(cands + (size_t)p * L * G * sp, prev, A, B, D, M, M_scalar, L, S, E, G, sp, alpha, beta, gamma,
                         out + (size_t)p * 5, NULL);
}

/* a7  Move deltas BY FULL RE-EVALUATION of the affected layer (BASELINE.json: "swap deltas
 *     equal full re-evaluation"): a move (l, a, b) exchanges the contents of slots a and b
 *     of layer l; the objective is a sum over layers, so only layer l's terms change.
 *     delta[5] = {dJ, dC_load, dC_comm, dC_mig, dmaxload}; NaN if the moved placement is
 *     invalid (an expert twice on one rank).  No closed form is used here.                */
void oracle_move_deltas(const int16_t *cur /*[L,NS]*/, const int16_t *prev /*[L,NS]*/,
                        const int32_t *moves /*[n,3]*/, int64_t n,
                        const double *A, const double *B, const double *D, const double *M, double M_scalar,
                        int L, int S, int E, int G, int sp, double alpha, double beta, double gamma,
                        double *delta /*[n,5]*/)
{
    const int NS = G * sp;
    (void)L;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        int l = moves[i * 3 + 0], a = moves[i * 3 + 1], b = moves[i * 3 + 2];
        int16_t *tmp = (int16_t *)malloc(sizeof(int16_t) * NS);
        memcpy(tmp, cur + (size_t)l * NS, sizeof(int16_t) * NS);
        int16_t v = tmp[a]; tmp[a] = tmp[b]; tmp[b] = v;
        double o0[5], o1[5], pl0[4], pl1[4];
        const double *Ml = M ? M + (size_t)l * E * G : NULL;
        int ok0 = oracle_objective(cur + (size_t)l * NS, prev + (size_t)l * NS, A + (size_t)l * S * E, B + (size_t)l * E, D, Ml, M_scalar,
                                   1, S, E, G, sp, alpha, beta, gamma, o0, pl0);
        int ok1 = oracle_objective(tmp, prev + (size_t)l * NS, A + (size_t)l * S * E, B + (size_t)l * E, D, Ml, M_scalar,
                                   1, S, E, G, sp, alpha, beta, gamma, o1, pl1);
        for (int j = 0; j < 5; ++j) delta[i * 5 + j] = (ok0 && ok1) ? o1[j] - o0[j] : NAN;
        free(tmp);
    }
}

/* ------------------------------------------------------------------------------------ */
/* Brute force over ALL placements of E experts onto G ranks x sp slots (NS == E, no
 * replicas), one layer: E!/(sp!)^G placements (tiny config: 16!/(4!)^4 = 63,063,000).
 * Enumerates expert -> rank assignments with capacity, evaluates each with
 * oracle_objective, returns the count, the minimum J and the first minimiser.           */
/* ------------------------------------------------------------------------------------ */
typedef struct {
    int E, G, sp, S;
    const int16_t *prev; const double *A, *B, *D, *M; double M_scalar, alpha, beta, gamma;
    int64_t count; double best; int16_t *best_place; int *rank_of; int *fill;
} bf_ctx;

static void bf_eval(bf_ctx *c)
{
    int16_t place[1024]; int pos[256];
    for (int g = 0; g < c->G; ++g) pos[g] = 0;
    for (int e = 0; e < c->E; ++e) { int g = c->rank_of[e]; place[g * c->sp + pos[g]++] = (int16_t)e; }
    double out[5];
    oracle_objective(place, c->prev, c->A, c->B, c->D, c->M, c->M_scalar, 1, c->S, c->E, c->G, c->sp,
                     c->alpha, c->beta, c->gamma, out, NULL);
    c->count++;
    if (out[0] < c->best) { c->best = out[0]; memcpy(c->best_place, place, sizeof(int16_t) * c->E); }
}

static void bf_rec(bf_ctx *c, int e)
{
    if (e == c->E) { bf_eval(c); return; }
    for (int g = 0; g < c->G; ++g) {
        if (c->fill[g] == c->sp) continue;
        c->fill[g]++; c->rank_of[e] = g;
        bf_rec(c, e + 1);
        c->fill[g]--;
    }
}

int64_t oracle_bruteforce(const int16_t *prev /*[NS]*/, const double *A /*[S,E]*/, const double *B /*[E]*/,
                          const double *D /*[S,G]*/, const double *M /*[E,G] or NULL*/, double M_scalar,
                          int S, int E, int G, int sp, double alpha, double beta, double gamma,
                          double *best_J, int16_t *best_place /*[NS]*/)
{
    /* split the search on the ranks of the first two experts so OpenMP has G*G branches;
       branches are merged in enumeration order so the FIRST minimiser wins. */
    const int nb = G * G;
    int64_t *cnt = (int64_t *)calloc(nb, sizeof(int64_t));
    double *bj = (double *)malloc(sizeof(double) * nb);
    int16_t *bp = (int16_t *)malloc(sizeof(int16_t) * (size_t)nb * E);
#pragma omp parallel for schedule(dynamic, 1)
    for (int br = 0; br < nb; ++br) {
        int rank_of[256], fill[256];
        for (int g = 0; g < G; ++g) fill[g] = 0;
        bf_ctx c = {E, G, sp, S, prev, A, B, D, M, M_scalar, alpha, beta, gamma, 0, INFINITY, bp + (size_t)br * E, rank_of, fill};
        int g0 = br / G, g1 = br % G;
        bj[br] = INFINITY;
        if (E < 2) { if (br == 0) { bf_rec(&c, 0); } }
        else {
            fill[g0]++; rank_of[0] = g0;
            if (fill[g1] < sp) { fill[g1]++; rank_of[1] = g1; bf_rec(&c, 2); }
        }
        cnt[br] = c.count; bj[br] = c.best;
    }
    int64_t total = 0; *best_J = INFINITY;
    for (int br = 0; br < nb; ++br) {
        total += cnt[br];
        if (bj[br] < *best_J) { *best_J = bj[br]; memcpy(best_place, bp + (size_t)br * E, sizeof(int16_t) * E); }
    }
    free(cnt); free(bj); free(bp);
    return total;
}

/* ------------------------------------------------------------------------------------ */
/* NEXT-1  The online greedy placement heuristic (section 5.3), step by step
 *     in the paper's order, one layer at a time (layers are independent):
 *       1. "ranks experts by a hotness signal derived from aggregate expert load and
 *          source-aware activation volume": hot[e] = (B[l,e] + sum_s A[l,s,e]) / r[l,e]
 *          (R17); the items are the slot contents of x0 (an expert hosted by r ranks
 *          is r items, each carrying 1/r of its tokens, R12), ordered by (hot descending,
 *          expert ascending, slot index in x0 ascending).
 *       2. "For each hot expert, ... enumerates feasible ranks that still have placement
 *          capacity and computes a local placement score"
 *              S[l,e,g] = alpha*Ccomm + beta*Cload + gamma*Cmig
 *          with (R17)  Ccomm = sum_s A[l,s,e] D[s,g] / r   "communication cost if expert e is
 *                              placed on rank g",
 *                      Cload = Lcur[g] + B[l,e]/r           "the resulting rank-load": load
 *                              already placed on g in this pass plus the item's,
 *                      Cmig  = M[l,e,g] if x0 does not host e on g, else 0  "relative to the
 *                              current placement".
 *          A rank is feasible when it has a free slot and does not already hold this expert.
 *       3. "assigns each expert to the feasible rank with the lowest score, breaking ties by
 *          preferring placements that avoid migration and then by choosing less-filled ranks"
 *          (PAPER.md:266-268); a last tie goes to the lowest rank index.
 *     All arithmetic is IEEE double, one operation at a time, in the order written here
 *     (S = ((alpha*Ccomm) + (beta*Cload)) + (gamma*Cmig), Ccomm summed over s ascending then
 *     divided by r); the decision precision of the contract is this double arithmetic.
 *     out[l, g*sp + i] = the i-th item assigned to rank g.  A layer whose x0 is invalid, or in
 *     which an item finds no feasible rank, gets a row of -1 (return value 0); the other
 *     layers are unaffected.                                                              */
/* ------------------------------------------------------------------------------------ */
int oracle_greedy_place(const int16_t *prev /*[L,NS]*/, const double *A /*[L,S,E]*/, const double *B /*[L,E]*/,
                        const double *D /*[S,G]*/, const double *M /*[L,E,G] or NULL*/, double M_scalar,
                        int L, int S, int E, int G, int sp, double alpha, double beta, double gamma,
                        int16_t *out /*[L,NS]*/)
{
    const int NS = G * sp;
    int ok = 1;
    double *x0 = (double *)malloc(sizeof(double) * (size_t)E * G), *r = (double *)malloc(sizeof(double) * E);
    double *hot = (double *)malloc(sizeof(double) * NS), *Lcur = (double *)malloc(sizeof(double) * G);
    int *order = (int *)malloc(sizeof(int) * NS), *fill = (int *)malloc(sizeof(int) * G);
    char *has = (char *)malloc((size_t)E * G);
    for (int i = 0; i < L * NS; ++i) out[i] = -1;
    for (int l = 0; l < L; ++l) {
        const int16_t *pv = prev + (size_t)l * NS;
        const double *Al = A + (size_t)l * S * E, *Bl = B + (size_t)l * E;
        int lok = 1;
        if (!build_x(pv, E, G, sp, x0, r)) { ok = 0; continue; }
        /* 1. hotness ranking of the items (selection sort on the total order) */
        for (int j = 0; j < NS; ++j) {
            int e = pv[j];
            double vol = 0.0;
            for (int s = 0; s < S; ++s) vol += Al[(size_t)s * E + e];
            hot[j] = (Bl[e] + vol) / r[e];
            order[j] = j;
        }
        for (int i = 0; i < NS; ++i) {
            int best = i;
            for (int j = i + 1; j < NS; ++j) {
                int a = order[j], b = order[best];
                int before_ = hot[a] > hot[b] || (hot[a] == hot[b] && (pv[a] < pv[b] || (pv[a] == pv[b] && a < b)));
                if (before_) best = j;
            }
            int t = order[i]; order[i] = order[best]; order[best] = t;
        }
        /* 2.-3. greedy assignment */
        for (int g = 0; g < G; ++g) { Lcur[g] = 0.0; fill[g] = 0; }
        memset(has, 0, (size_t)E * G);
        for (int i = 0; i < NS && lok; ++i) {
            int e = pv[order[i]];
            double b = Bl[e] / r[e];
            int bg = -1, bmig = 0, bfill = 0; double bs = 0.0;
            for (int g = 0; g < G; ++g) {
                if (fill[g] >= sp || has[(size_t)e * G + g]) continue;
                double c = 0.0;
                for (int s = 0; s < S; ++s) c += Al[(size_t)s * E + e] * D[(size_t)s * G + g];
                c = c / r[e];
                int mig = x0[(size_t)e * G + g] == 0.0;
                double m = mig ? (M ? M[((size_t)l * E + e) * G + g] : M_scalar) : 0.0;
                double load = Lcur[g] + b;
                double sc = ((alpha * c) + (beta * load)) + (gamma * m);
                int better = bg < 0 || sc < bs || (sc == bs && (mig < bmig || (mig == bmig && fill[g] < bfill)));
                if (better) { bg = g; bs = sc; bmig = mig; bfill = fill[g]; }
            }
            if (bg < 0) { lok = 0; break; }
            out[(size_t)l * NS + bg * sp + fill[bg]] = (int16_t)e;
            fill[bg]++; has[(size_t)e * G + bg] = 1; Lcur[bg] += b;
        }
        if (!lok) { ok = 0; for (int j = 0; j < NS; ++j) out[(size_t)l * NS + j] = -1; }
    }
    free(x0); free(r); free(hot); free(Lcur); free(order); free(fill); free(has);
    return ok;
}

/* ------------------------------------------------------------------------------------ */
/* NEXT-3  Expert mapping, logical -> physical ("fuse source counting with expert mapping",
 *     PAPER.md:276, 368; R18): under placement `place` (slot -> expert) the slots
 *     hosting expert e, in ascending order, are s_0 < ... < s_{r-1}; the choice (t, j) with
 *     ids[t,j] = e goes to slot s_{t mod r} (t = token index in the step).  r = 1 in the paper.
 *     phys[t,j] = -1 when no slot hosts e.                                                 */
/* ------------------------------------------------------------------------------------ */
void oracle_expert_map(const int32_t *ids /*[T,k]*/, const int16_t *place /*[NS]*/, int T, int k, int NS,
                       int32_t *phys /*[T,k]*/)
{
    for (int t = 0; t < T; ++t)
        for (int j = 0; j < k; ++j) {
            int e = ids[(size_t)t * k + j], r = 0, pick = -1;
            for (int s = 0; s < NS; ++s) r += (place[s] == e);
            if (r > 0) {
                int want = t % r, seen = 0;
                for (int s = 0; s < NS; ++s)
                    if (place[s] == e) { if (seen == want) { pick = s; break; } ++seen; }
            }
            phys[(size_t)t * k + j] = pick;
        }
}

/* ------------------------------------------------------------------------------------ */
/* NEXT-2  Algorithm 1, Global DP Engine Scheduling (section 4.3), for one
 *     scheduler instance and a sequence of R incoming requests, in the algorithm's order.
 *     The extracted listing lost some step numbers; the steps are
 *     unambiguous.  Undefined pieces take the readings of DESIGN.md R19:
 *       HighKV(kv)  = kv > high_kv          (90 %)
 *       LargeGap(d) = d  > large_gap        (10 %)
 *       P_kv(kv)    = lambda_kv  * kv       token-equivalent penalties, linear;
 *       P_moe(moe)  = lambda_moe * moe      moe is the relative MoE pressure (mean 1)
 *       CLOSE(D, r) = D < close_frac * len(r)
 *       Next(E)     = engine rr, then rr <- (rr + 1) mod N (ordered dispatch)
 *       compensation: after a request is assigned, comp[e*] += len(r), "a
 *       temporary pressure estimate" that lasts until the caller loads a fresh trace.
 *     trace[n] = {kv, pre_rem, wait, moe}.  score = (((pre_rem + wait) + comp) + lambda_kv*kv)
 *     + lambda_moe*moe in IEEE double, one rounding per operation; argmin over the
 *     lexicographic key (score, kv, i).  argmin / argmax of kv: lowest index.  */
/* ------------------------------------------------------------------------------------ */
void oracle_select_engines(const float *trace /*[N,4]*/, int complete, const float *req_len /*[R]*/, int N, int R,
                           double high_kv, double large_gap, double lambda_kv, double lambda_moe, double close_frac,
                           double *comp /*[N] inout*/, int32_t *rr /*[1] inout*/, int32_t *engine /*[R]*/)
{
    *rr = ((*rr % N) + N) % N;                              /* Next(E) counts modulo N (R19) */
    for (int q = 0; q < R; ++q) {
        double len = (double)req_len[q];
        int pick = -1;
        if (!complete) {                                   /* line 1-2: traces incomplete -> ordered dispatch */
            pick = *rr; *rr = (*rr + 1) % N;
        } else {
            int imin = 0, imax = 0;                        /* line 6 */
            for (int i = 1; i < N; ++i) {
                if (trace[i * 4] < trace[imin * 4]) imin = i;
                if (trace[i * 4] > trace[imax * 4]) imax = i;
            }
            double kvmax = (double)trace[imax * 4], kvmin = (double)trace[imin * 4];
            if (kvmax > high_kv && (kvmax - kvmin) > large_gap) {      /* line 7-8 */
                pick = imin;
            } else {
                double smin = 0.0, smax = 0.0; int best = 0; double bs = 0.0, bkv = 0.0;
                for (int i = 0; i < N; ++i) {              /* line 10-12 */
                    double kv = (double)trace[i * 4], pre = (double)trace[i * 4 + 1], wait = (double)trace[i * 4 + 2],
                           moe = (double)trace[i * 4 + 3];
                    double sc = (((pre + wait) + comp[i]) + (lambda_kv * kv)) + (lambda_moe * moe);
                    if (i == 0 || sc < smin) smin = sc;
                    if (i == 0 || sc > smax) smax = sc;
                    if (i == 0 || sc < bs || (sc == bs && kv < bkv)) { best = i; bs = sc; bkv = kv; }
                }
                double delta = smax - smin;                /* line 13 */
                if (delta < close_frac * len) {            /* line 14-15 */
                    pick = *rr; *rr = (*rr + 1) % N;
                } else {
                    pick = best;                           /* line 17 */
                }
            }
        }
        engine[q] = pick;
        comp[pick] += len;                                 /* compensation */
    }
}

/* ------------------------------------------------------------------------------------ */
/* Algorithm 2, Request Scheduler with SJF and Aging (section 4.4; the
 *     extracted listing is scrambled, R20): for every request r of the waiting queue,
 *     waiting time w_r = now - arrival_r; if w_r >= theta_age the request gets high priority,
 *     otherwise its priority is its prefill length; the queue is sorted by priority ascending.
 *     Reading R20 for what the paper leaves open: aged requests come first, oldest first; the
 *     others by prefill length (shortest first), equal lengths oldest first; a last tie goes to
 *     the position in the input queue.  order[i] = input position of the i-th request to run.   */
/* ------------------------------------------------------------------------------------ */
static float alg2_arrival(const float *arrival, int a)
{
    return arrival[a] != arrival[a] ? INFINITY : arrival[a];      /* a NaN arrival is the youngest request (R20) */
}

static int alg2_before(const float *arrival, const int32_t *prefill, float now, float theta, int a, int b)
{
    float ta = alg2_arrival(arrival, a), tb = alg2_arrival(arrival, b);
    int aged_a = (now - ta) >= theta, aged_b = (now - tb) >= theta;
    if (aged_a != aged_b) return aged_a;                        /* high priority first */
    if (!aged_a && prefill[a] != prefill[b]) return prefill[a] < prefill[b];
    if (ta != tb) return ta < tb;
    return a < b;
}

void oracle_order_queue(const float *arrival /*[n]*/, const int32_t *prefill /*[n]*/, int n, float now, float theta_age,
                        int32_t *order /*[n]*/)
{
    for (int i = 0; i < n; ++i) order[i] = i;
    for (int i = 1; i < n; ++i) {                               /* insertion sort under the total order */
        int x = order[i], j = i - 1;
        while (j >= 0 && alg2_before(arrival, prefill, now, theta_age, x, order[j])) { order[j + 1] = order[j]; --j; }
        order[j + 1] = x;
    }
}

/* ------------------------------------------------------------------------------------ */
/* Swap-based refinement of a placement (the local search SURVEY.md section 8f attaches to
 *     NEXT-1; not in the paper, R21): `iters` rounds; in each round and each layer
 *     the best single slot exchange (lowest dJ by FULL re-evaluation, canonical order a < b,
 *     first on ties, invalid moves skipped) is applied when
 *         dJ < -1e-4 * (alpha*|dC_comm| + beta*|dC_load| + gamma*|dC_mig|)
 *     (a margin above rounding so that the fp32 kernel and this fp64 text cannot cycle on
 *     noise).  cur is updated in place; applied[l] counts the exchanges of layer l.          */
/* ------------------------------------------------------------------------------------ */
void oracle_refine(int16_t *cur /*[L,NS] inout*/, const int16_t *prev, const double *A, const double *B, const double *D,
                   const double *M, double M_scalar, int L, int S, int E, int G, int sp,
                   double alpha, double beta, double gamma, int iters, int32_t *applied /*[L]*/)
{
    const int NS = G * sp;
    const int64_t npairs = (int64_t)NS * (NS - 1) / 2;
    int32_t *mv = (int32_t *)malloc(sizeof(int32_t) * 3 * (size_t)npairs);
    double *dl = (double *)malloc(sizeof(double) * 5 * (size_t)npairs);
    for (int l = 0; l < L; ++l) applied[l] = 0;
    for (int it = 0; it < iters; ++it)
        for (int l = 0; l < L; ++l) {
            int64_t q = 0;
            for (int a = 0; a < NS; ++a)
                for (int b = a + 1; b < NS; ++b) { mv[q * 3] = l; mv[q * 3 + 1] = a; mv[q * 3 + 2] = b; ++q; }
            oracle_move_deltas(cur, prev, mv, npairs, A, B, D, M, M_scalar, L, S, E, G, sp, alpha, beta, gamma, dl);
            int64_t best = -1;
            for (int64_t i = 0; i < npairs; ++i) {
                if (dl[i * 5] != dl[i * 5]) continue;
                if (best < 0 || dl[i * 5] < dl[best * 5]) best = i;
            }
            if (best < 0) continue;
            double thr = 1e-4 * (alpha * fabs(dl[best * 5 + 2]) + beta * fabs(dl[best * 5 + 1]) + gamma * fabs(dl[best * 5 + 3]));
            if (dl[best * 5] < -thr) {
                int a = mv[best * 3 + 1], b = mv[best * 3 + 2];
                int16_t t = cur[(size_t)l * NS + a]; cur[(size_t)l * NS + a] = cur[(size_t)l * NS + b]; cur[(size_t)l * NS + b] = t;
                applied[l]++;
            }
        }
    free(mv); free(dl);
}

/* threads the OpenMP loops above will use (reported as cpu_baseline.cores by bench.py) */
#ifdef _OPENMP
#include <omp.h>
int oracle_num_threads(void) { return omp_get_max_threads(); }
/* bench.py times the same code on one thread as well; no arithmetic depends on it */
void oracle_set_num_threads(int n) { if (n > 0) omp_set_num_threads(n); }
#else
int oracle_num_threads(void) { return 1; }
void oracle_set_num_threads(int n) { (void)n; }
#endif
