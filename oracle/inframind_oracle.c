/*
 * inframind_oracle.c — plain, slow, single-purpose CPU ORACLE for the INFRAMIND CMDP rollout + returns.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, link or call it.  It shares no code, header, table
 * generator or helper with the CUDA path (paper_2606_11440_b200/csrc); the struct definitions below are
 * typed independently from include/inframind.h.
 *
 * What it computes.  The paper fixes the MDP's interfaces: executor state
 * (Eq. 1), joint action decode m = a div 3, sigma = a mod 3, cost
 * C_k = l_k/beta and reward R in {0,1} (Eq. 2), Lagrangian r - lambda*C (PAPER.md:76-79,
 * Eq. 3), planner outputs (tau, K, roles), deadline = t_arrive + beta inherited by every
 * call and EDF per model queue, planner utility U_i, and the mean
 * constraint violation C-bar of the dual update (Eq. 7).  The paper trains on a live
 * vLLM pool and has no simulator; the tick semantics are the numbered Readings R1..R34 of DESIGN.md
 * (from SURVEY.md §8(c)), which this file follows STEP BY STEP in the canonical order, loops ascending,
 * with no blocking, fusion or reordering.  Requests are the calls (query, agent) and live in a table indexed
 * by query*4 + agent; a RUNNING request holds a slot of its model (R10) and its service draw is keyed by that
 * slot (R2, R11).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known answers (P1), Poisson/budget/lognormal
 * tables (P2-P4), M/M/1 mean sojourn 1/(mu-lambda) (P6), Little's law (P7), conservation (P8), EDF
 * brute force (P9), action decode (P10), sampler closed forms (P11), MLP vs float64 numpy (P12), GAE
 * vs direct discounted sum (P13), Lagrangian linearity (P14), determinism / split / E-invariance (P15),
 * utility normalisation (P17), deterministic stamps (P18), preemption (P19), service rate (P20); and
 * (tests/test_oracle_pins2.py) the cost value l/beta per call, the success bit and its OR
 * composition (R18/R19), the debate / review stage tables and K_eff (R17), the head-of-line stop under a KV
 * misfit (R21), the episode hard reset (R33) and the near-boundary window (R25).
 * PARITY UNPINNED (definitional readings with no external truth): role semantics (R16),
 * feature scale constants (R14-15), drop penalty (R9), snapshot staleness (R14).
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/oracle.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAXN 16
#define ORC_DT_US 50000u

/* ------------------------------------------------------------------------------------------- spec */
typedef struct {
    uint32_t rate_tok_s, slots, kv_cap, prefill_us_per_ktok;
    uint32_t succ_thresh[3];
    float kv_inv;
} orc_model;

typedef struct {
    uint32_t n_models, qcap, rcap, max_ticks;
    uint32_t sched_mode, kv_preempt, cost_mode, episode_ticks;
    uint32_t budget_norm_ticks, n_levels, policy_dtype, f_in;
    uint32_t hidden, in_tok_const, mix_thresh, keep_logits;
    uint32_t depth_median_tok[3];
    uint32_t mix_lo[2], mix_hi[2];
    orc_model model[ORC_MAXN];
    const uint32_t *out_tok_mult_q16; /* [1024] */
    const uint32_t *in_tok_table;     /* [1024] or NULL */
    const uint32_t *arr_cdf;          /* [n_levels][32] */
} orc_spec;

/* forced decisions: the GPU's log, sorted by (env_local, tick, query, agent), one set per kind */
typedef struct {
    const int64_t *off;      /* [n_envs+1] record range of each local env */
    const int32_t *t;        /* absolute tick */
    const uint16_t *q;
    const uint8_t *agent;
    const uint32_t *payload; /* GPU action (exec) or packed plan */
    const float *logits;     /* [n][n_out] or NULL */
} orc_forced_kind;

typedef struct {
    orc_forced_kind plan, exec;
} orc_forced;

/* ------------------------------------------------------------------------------------------ state */
enum { ST_FREE = 0, ST_WAIT = 1, ST_RUN = 2 };
enum { TOPO_SINGLE = 0, TOPO_CHAIN = 1, TOPO_DEBATE = 2, TOPO_REVIEW = 3 };
enum { STREAM_ARR = 1, STREAM_QRY = 2, STREAM_PLAN = 3, STREAM_EXEC = 4, STREAM_SVC = 5 };
enum { C_ARRIVALS, C_DROPPED, C_FINISHED, C_SOLVED, C_MISSED, C_ISSUED, C_CALLS_DONE, C_PREEMPT,
       C_SUM_SOJOURN, C_SUM_LIVE_MID, C_PLANS, C_EXEC_DEC, C_SUM_RUNNING, C_SUM_WAITING, C_NEAR, C_ABANDONED, C_N };

typedef struct {
    uint8_t live, planned, topo, cnt, keff, stage, n_stages, pending, succ;
    uint8_t roles[4];
    int32_t arrive, deadline;
    uint32_t budget, in_tok;
} oq_t;

/* R10: a request is the call (query, agent); the table is indexed by query*4 + agent.  A RUNNING request
 * occupies one of the S_k slots of its model (north_star (1): "per-model slots"). */
typedef struct {
    uint8_t state, model, depth, agent, succ, slot;
    uint16_t query;
    int32_t deadline, issue;
    uint32_t remaining, out_total, prefill_us, in_tok;
} or_t;

typedef struct {
    uint32_t n_wait, n_run, kv_used, ewma_q8;
} om_t;

typedef struct {
    int32_t t;
    uint16_t q;
    uint8_t agent, pad;
    uint32_t payload;
    float logp, value;
} odec_t;

typedef struct {
    uint32_t env, info;
    int32_t arrive;
    uint32_t sojourn;
} oqlog_t;

typedef struct {
    oq_t *q;
    or_t *r;
    om_t m[ORC_MAXN];
    uint64_t ctr[C_N];
    odec_t *plan_log, *exec_log;
    float *plan_logits, *exec_logits;
    size_t n_plan, cap_plan, n_exec, cap_exec;
    oqlog_t *qlog;
    size_t n_qlog, cap_qlog;
    /* lock-step statistics */
    uint64_t n_desync, n_hard, n_near;
    double max_logit_diff, max_value_diff;
    size_t cur_plan, cur_exec; /* cursors into the forced logs */
} oenv_t;

typedef struct {
    const float *W1, *b1, *W2, *b2, *W3, *b3; /* fp32 views (bf16 widened exactly at load) */
    uint32_t n_out;
} onet_t;

typedef struct orc_ctx {
    orc_spec s;
    uint32_t n_envs;
    uint32_t *env_id;
    uint8_t *env_level;
    uint64_t seed;
    int32_t tick;            /* absolute tick of the next rollout's first tick */
    uint32_t last_T;         /* ticks of the last rollout */
    oenv_t *env;
    uint32_t *tab_mult, *tab_intok, *tab_cdf;
    float *rew, *cost, *val; /* [max_ticks+1][n_envs] */
    uint8_t *done, *miss;
    double *adv, *ret;
    int have_returns;
    double cbar, ubar, usigma, sum_cost;
    uint64_t n_final;
    float *wbuf;             /* decoded weights */
    onet_t plan, exec;
    const orc_forced *forced;
} orc_ctx;

/* ------------------------------------------------------------------------ R2: Philox4x32-10 */
/* Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3" (SC'11): multipliers
 * 0xD2511F53 / 0xCD9E8D57, Weyl key increments 0x9E3779B9 / 0xBB67AE85, 10 rounds. */
typedef struct { uint32_t v[4]; } ph4;

ph4 orc_philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1)
{
    for (int r = 0; r < 10; r++) {
        if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    ph4 o = {{c0, c1, c2, c3}};
    return o;
}

/* R2: key = (seed_lo, seed_hi ^ stream), counter = (env, tick, slot, sub) with the GLOBAL env id */
static ph4 draw(const orc_ctx *c, uint32_t stream, uint32_t gid, int32_t t, uint32_t slot, uint32_t sub)
{
    return orc_philox4x32_10(gid, (uint32_t)t, slot, sub, (uint32_t)c->seed, (uint32_t)(c->seed >> 32) ^ stream);
}

static uint32_t mulhi32(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a * b) >> 32); }

/* R3: policy uniform u = (x>>8) * 2^-24 in [0,1), exact in fp32 */
static float u24(uint32_t x) { return (float)(x >> 8) * 0x1p-24f; }

/* -------------------------------------------------------------------- R23: im_exp / im_tanh */
/* A DEFINED function (typed independently on the GPU side).  x <= 0 expected by callers. */
float orc_im_exp(float x)
{
    if (x < -80.0f) return 0.0f;
    float n = rintf(x * 0x1.715476p+0f);            /* log2(e) rounded to fp32 */
    float r = fmaf(n, -0x1.62e400p-1f, x);          /* Cody-Waite, ln2 = hi + lo */
    r = fmaf(n, -0x1.7f7d1cp-20f, r);
    float p = 0x1.6c16c2p-10f;                      /* 1/720 */
    p = fmaf(p, r, 0x1.111112p-7f);                 /* 1/120 */
    p = fmaf(p, r, 0x1.555556p-5f);                 /* 1/24  */
    p = fmaf(p, r, 0x1.555556p-3f);                 /* 1/6   */
    p = fmaf(p, r, 0.5f);
    p = fmaf(p, r, 1.0f);
    p = fmaf(p, r, 1.0f);
    return ldexpf(p, (int)n);
}

float orc_im_tanh(float x)
{
    float e = orc_im_exp(-2.0f * fabsf(x));
    float num = 1.0f - e, den = 1.0f + e;
    return copysignf(num / den, x);
}

/* ------------------------------------------------------------------------------ R24: sampler */
/* m = max l; e_i = im_exp(l_i - m); c_i = c_{i-1} + e_i (ascending, plain fp32); Z = c_{n-1};
 * th = u*Z; a = first i with c_i > th else n-1; logp = (l_a - m) - logf(Z). c[] returned for checks */
uint32_t orc_sample(const float *l, uint32_t n, float u, float *logp, float *cdf_out)
{
    float m = l[0];
    for (uint32_t i = 1; i < n; i++) if (l[i] > m) m = l[i];
    float c[64];
    float acc = 0.0f;
    for (uint32_t i = 0; i < n; i++) { acc = acc + orc_im_exp(l[i] - m); c[i] = acc; }
    float Z = c[n - 1];
    float th = u * Z;
    uint32_t a = n - 1;
    for (uint32_t i = 0; i < n; i++) if (c[i] > th) { a = i; break; }
    if (logp) *logp = (l[a] - m) - logf(Z);
    if (cdf_out) for (uint32_t i = 0; i < n; i++) cdf_out[i] = c[i];
    return a;
}

/* near-boundary rule (north_star; R25(3)): action `a` is acceptable iff u lies within 1e-6 of its
 * CDF interval [c_{a-1}/Z, c_a/Z). */
static int near_ok(const float *c, uint32_t n, float u, uint32_t a)
{
    double Z = c[n - 1];
    double lo = (a == 0) ? 0.0 : (double)c[a - 1] / Z;
    double hi = (a == n - 1) ? 1.0 : (double)c[a] / Z;
    return ((double)u >= lo - 1e-6) && ((double)u <= hi + 1e-6);
}

/* exported for its pin (tests/test_oracle_pins2.py): the same function, callable */
int orc_near_ok(const float *c, uint32_t n, float u, uint32_t a) { return near_ok(c, n, u, a); }

/* --------------------------------------------------------------------------- R22 / R25: MLP */
static float bf16_round(float x) /* RNE to bf16, returned as fp32 */
{
    uint32_t u; memcpy(&u, &x, 4);
    uint32_t r = ((u >> 16) & 1u) + 0x7FFFu;
    u = (u + r) & 0xFFFF0000u;
    float y; memcpy(&y, &u, 4);
    return y;
}

/* fp32 contract R22: y_o = b_o; for k ascending: y_o = fmaf(W[o][k], x_k, y_o); hidden = im_tanh(y).
 * bf16 contract R25: layer inputs rounded to bf16 (RNE), weights already bf16, exact products summed
 * in double (the limit of "fp32 accumulation in unspecified order"), fp32 bias, tanh in double. */
static void mlp_forward(const orc_ctx *c, const onet_t *net, const float *x, float *out)
{
    const uint32_t F = c->s.f_in, H = c->s.hidden;
    float h1[512], h2[512], xin[512];
    if (c->s.policy_dtype == 0) {
        for (uint32_t o = 0; o < H; o++) {
            float y = net->b1[o];
            for (uint32_t k = 0; k < F; k++) y = fmaf(net->W1[o * F + k], x[k], y);
            h1[o] = orc_im_tanh(y);
        }
        for (uint32_t o = 0; o < H; o++) {
            float y = net->b2[o];
            for (uint32_t k = 0; k < H; k++) y = fmaf(net->W2[o * H + k], h1[k], y);
            h2[o] = orc_im_tanh(y);
        }
        for (uint32_t o = 0; o < net->n_out; o++) {
            float y = net->b3[o];
            for (uint32_t k = 0; k < H; k++) y = fmaf(net->W3[o * H + k], h2[k], y);
            out[o] = y;
        }
    } else {
        for (uint32_t k = 0; k < F; k++) xin[k] = bf16_round(x[k]);
        for (uint32_t o = 0; o < H; o++) {
            double y = net->b1[o];
            for (uint32_t k = 0; k < F; k++) y += (double)net->W1[o * F + k] * (double)xin[k];
            h1[o] = bf16_round((float)tanh(y));
        }
        for (uint32_t o = 0; o < H; o++) {
            double y = net->b2[o];
            for (uint32_t k = 0; k < H; k++) y += (double)net->W2[o * H + k] * (double)h1[k];
            h2[o] = bf16_round((float)tanh(y));
        }
        for (uint32_t o = 0; o < net->n_out; o++) {
            double y = net->b3[o];
            for (uint32_t k = 0; k < H; k++) y += (double)net->W3[o * H + k] * (double)h2[k];
            out[o] = (float)y;
        }
    }
}

/* exported for the P12 pin */
int orc_mlp_forward(const orc_ctx *c, int which, const float *x, float *out)
{
    mlp_forward(c, which ? &c->exec : &c->plan, x, out);
    return 0;
}

/* ---------------------------------------------------------------------------- weight blob R26 */
static size_t pad16(size_t n) { return (n + 15u) & ~(size_t)15u; }

static int load_blob(orc_ctx *c, const uint8_t *blob)
{
    const uint32_t *h = (const uint32_t *)blob;
    const uint32_t F = c->s.f_in, H = c->s.hidden, N = c->s.n_models;
    if (h[0] != 0x494D5042u || h[1] != c->s.policy_dtype || h[2] != F || h[3] != H || h[4] != 24 || h[5] != 3 * N + 1) return -2;
    size_t total = 2 * ((size_t)H * F + H + (size_t)H * H + H) + (size_t)(24 + 3 * N + 1) * (H + 1);
    free(c->wbuf);
    c->wbuf = (float *)malloc(total * sizeof(float));
    float *w = c->wbuf;
    const uint8_t *p = blob + 32;
    const int bf = c->s.policy_dtype == 1;
    for (int net = 0; net < 2; net++) {
        onet_t *o = net ? &c->exec : &c->plan;
        o->n_out = net ? 3 * N + 1 : 24;
        size_t shapes[6] = {(size_t)H * F, H, (size_t)H * H, H, (size_t)o->n_out * H, o->n_out};
        const float **dst[6] = {&o->W1, &o->b1, &o->W2, &o->b2, &o->W3, &o->b3};
        for (int a = 0; a < 6; a++) {
            size_t n = shapes[a];
            int is_w = (a % 2 == 0);
            *dst[a] = w;
            if (is_w && bf) {
                const uint16_t *s = (const uint16_t *)p;
                for (size_t i = 0; i < n; i++) { uint32_t u = (uint32_t)s[i] << 16; memcpy(&w[i], &u, 4); }
                p += pad16(2 * n);
            } else {
                memcpy(w, p, 4 * n);
                p += pad16(4 * n);
            }
            w += n;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------ topologies R17 */
/* single [1]; chain [1,1,...] (K stages); debate [K-1 parallel, 1 judge]; review [1 writer, K-1 parallel] */
static uint32_t keff_of(uint32_t topo, uint32_t K)
{
    if (topo == TOPO_SINGLE) return 1;
    if (topo == TOPO_CHAIN) return K;
    return K < 2 ? 2 : K;
}
static uint32_t n_stages_of(uint32_t topo, uint32_t keff)
{
    if (topo == TOPO_SINGLE) return 1;
    if (topo == TOPO_CHAIN) return keff;
    return 2;
}
static void stage_calls(uint32_t topo, uint32_t keff, uint32_t stage, uint32_t *first_agent, uint32_t *n_calls)
{
    if (topo == TOPO_SINGLE) { *first_agent = 0; *n_calls = 1; }
    else if (topo == TOPO_CHAIN) { *first_agent = stage; *n_calls = 1; }
    else if (topo == TOPO_DEBATE) {
        if (stage == 0) { *first_agent = 0; *n_calls = keff - 1; } else { *first_agent = keff - 1; *n_calls = 1; }
    } else {
        if (stage == 0) { *first_agent = 0; *n_calls = 1; } else { *first_agent = 1; *n_calls = keff - 1; }
    }
}

/* --------------------------------------------------------------------------------- features R15 */
static void shared_block(const orc_ctx *c, const om_t *snap, float b, uint32_t in_tok, float *x)
{
    const uint32_t N = c->s.n_models;
    memset(x, 0, sizeof(float) * c->s.f_in);
    x[0] = b;
    for (uint32_t k = 0; k < N; k++) {
        x[1 + k] = (float)snap[k].n_wait * 0x1p-6f;          /* d_queue (R14) */
        x[1 + N + k] = (float)snap[k].ewma_q8 * 0x1p-18f;    /* d_e2e: ticks/1024 */
        x[1 + 2 * N + k] = (float)snap[k].kv_used * c->s.model[k].kv_inv; /* d_kv */
    }
    x[3 * N + 1] = (float)in_tok * 0x1p-13f;
}

/* ----------------------------------------------------------------------------------- logging */
static void push_dec(odec_t **log, float **lg, size_t *n, size_t *cap, uint32_t n_out, int keep,
                     odec_t d, const float *logits)
{
    if (*n == *cap) {
        *cap = *cap ? *cap * 2 : 256;
        *log = (odec_t *)realloc(*log, *cap * sizeof(odec_t));
        if (keep) *lg = (float *)realloc(*lg, *cap * n_out * sizeof(float));
    }
    (*log)[*n] = d;
    if (keep) memcpy(*lg + *n * n_out, logits, n_out * sizeof(float));
    (*n)++;
}

static void stat_logits(oenv_t *E, const float *own, const float *gpu, uint32_t n)
{
    for (uint32_t i = 0; i < n; i++) {
        double d = fabs((double)own[i] - (double)gpu[i]);
        if (!(d <= E->max_logit_diff)) E->max_logit_diff = d; /* NaN-propagating */
    }
}

/* one softmax head decision, with teacher forcing / resync (R24, R25) */
static uint32_t decide_head(oenv_t *E, const float *own, const float *forced_logits, uint32_t n, float u,
                            int have_gpu_action, uint32_t gpu_action, float *logp)
{
    float cdf[64];
    const float *src = forced_logits ? forced_logits : own;
    uint32_t a = orc_sample(src, n, u, logp, cdf);
    if (have_gpu_action && gpu_action != a) {
        if (gpu_action < n && near_ok(cdf, n, u, gpu_action)) E->n_near++; else E->n_hard++;
        if (gpu_action < n) {       /* adopt the GPU's action: that IS the resync (R25) */
            a = gpu_action;
            float m = src[0];
            for (uint32_t i = 1; i < n; i++) if (src[i] > m) m = src[i];
            if (logp) *logp = (src[a] - m) - logf(cdf[n - 1]);
        }
    }
    return a;
}

/* -------------------------------------------------------------------------------- the tick */
static uint32_t lowest_free_query(const orc_ctx *c, const oenv_t *E)
{
    for (uint32_t i = 0; i < c->s.qcap; i++) if (!E->q[i].live) return i;
    return c->s.qcap;
}
static uint32_t n_req(const orc_ctx *c) { return 4u * c->s.qcap; }

/* R10: lowest free slot of model k (the slots taken are those of its RUNNING requests) */
static uint32_t lowest_free_slot(const orc_ctx *c, const oenv_t *E, uint32_t k)
{
    for (uint32_t sl = 0; sl < c->s.model[k].slots; sl++) {
        int taken = 0;
        for (uint32_t i = 0; i < n_req(c); i++)
            if (E->r[i].state == ST_RUN && E->r[i].model == k && E->r[i].slot == sl) taken = 1;
        if (!taken) return sl;
    }
    return c->s.model[k].slots;
}

/* R2: the slots of all models are numbered consecutively, each model's range padded to a multiple of 8, so
 * that one Philox call (8 sixteen-bit fields) serves 8 slots of one model */
static uint32_t global_slot(const orc_ctx *c, uint32_t k, uint32_t sl)
{
    uint32_t base = 0;
    for (uint32_t j = 0; j < k; j++) base += (c->s.model[j].slots + 7u) & ~7u;
    return base + sl;
}

/* R20: the queue of model k is ordered by (deadline, query*4+agent) (EDF) or by
 * (issue, query*4+agent) (FCFS); the pair is unique, so there is exactly one correct order.  Since
 * remaining budget = deadline - t, "earliest remaining budget first" at a fixed t is the same order. */
static int key_less(const orc_ctx *c, const or_t *a, uint32_t ia, const or_t *b, uint32_t ib)
{
    int32_t ka = c->s.sched_mode ? a->deadline : a->issue, kb = c->s.sched_mode ? b->deadline : b->issue;
    if (ka != kb) return ka < kb;
    return ia < ib;
}

static void env_tick(orc_ctx *c, uint32_t ei, int32_t t, uint32_t trow)
{
    const orc_spec *s = &c->s;
    oenv_t *E = &c->env[ei];
    const uint32_t gid = c->env_id[ei], N = s->n_models;
    uint32_t rew = 0, miss = 0;
    uint64_t cost_q16 = 0;
    float x[512], logits[64];

    /* ---- A ARRIVE (R5, R7, R8, R9) */
    {
        uint32_t xr = draw(c, STREAM_ARR, gid, t, 0, 0).v[0];
        const uint32_t *cdf = c->tab_cdf + 32u * c->env_level[ei];
        uint32_t n = 0;
        for (uint32_t j = 0; j < 31; j++) if (xr >= cdf[j]) n++;
        uint32_t nfree = 0;
        for (uint32_t i = 0; i < s->qcap; i++) if (!E->q[i].live) nfree++;
        uint32_t n_ok = n < nfree ? n : nfree;
        E->ctr[C_ARRIVALS] += n;
        E->ctr[C_DROPPED] += n - n_ok;
        miss += n - n_ok;                        /* R9: a dropped query is a miss ... */
        cost_q16 += (uint64_t)(n - n_ok) << 16;  /* ... with cost 1.0 and reward 0 */
        for (uint32_t j = 0; j < n_ok; j++) {
            uint32_t qi = lowest_free_query(c, E);
            ph4 d = draw(c, STREAM_QRY, gid, t, j, 0);
            uint32_t comp = d.v[2] < s->mix_thresh ? 0u : 1u;
            oq_t *q = &E->q[qi];
            memset(q, 0, sizeof(*q));
            q->live = 1;
            q->budget = s->mix_lo[comp] + mulhi32(d.v[0], s->mix_hi[comp] - s->mix_lo[comp] + 1u);
            q->in_tok = c->tab_intok ? c->tab_intok[d.v[1] >> 22] : s->in_tok_const;
            q->arrive = t;
            q->deadline = t + (int32_t)q->budget;  /* PAPER.md:117 deadline = t_arrive + beta */
        }
        uint32_t live = 0;
        for (uint32_t i = 0; i < s->qcap; i++) live += E->q[i].live;
        E->ctr[C_SUM_LIVE_MID] += live;
    }

    /* ---- B SNAPSHOT (R14): telemetry of the state left by tick t-1; critic V[t] (R30) */
    om_t snap[ORC_MAXN];
    memcpy(snap, E->m, sizeof(snap));
    shared_block(c, snap, 0.0f, 0, x);
    mlp_forward(c, &c->exec, x, logits);
    c->val[(size_t)trow * c->n_envs + ei] = logits[3 * N];

    const orc_forced *F = c->forced;

    /* ---- C PLAN (R15, R16): every query created in A, index ascending */
    for (uint32_t qi = 0; qi < s->qcap; qi++) {
        oq_t *q = &E->q[qi];
        if (!q->live || q->planned) continue;
        float b = (float)q->budget / (float)s->budget_norm_ticks;
        shared_block(c, snap, b, q->in_tok, x);
        mlp_forward(c, &c->plan, x, logits);
        ph4 d0 = draw(c, STREAM_PLAN, gid, t, qi, 0), d1 = draw(c, STREAM_PLAN, gid, t, qi, 1);
        const float *fl = NULL; int have = 0; uint32_t gp = 0;
        if (F && F->plan.off) {
            size_t cur = (size_t)F->plan.off[ei] + E->cur_plan;
            if (cur < (size_t)F->plan.off[ei + 1] && F->plan.t[cur] == t && F->plan.q[cur] == qi) {
                have = 1; gp = F->plan.payload[cur];
                if (F->plan.logits) { fl = F->plan.logits + cur * 24; stat_logits(E, logits, fl, 24); }
                E->cur_plan++;
            } else E->n_desync++;
        }
        float lp_t, lp_c, lp_r[4];
        uint32_t topo = decide_head(E, logits, fl, 4, u24(d0.v[0]), have, gp & 3u, &lp_t);
        uint32_t cnt = decide_head(E, logits + 4, fl ? fl + 4 : NULL, 4, u24(d0.v[1]), have, (gp >> 2) & 3u, &lp_c);
        uint32_t roles = 0;
        for (uint32_t a = 0; a < 4; a++) {
            uint32_t r = decide_head(E, logits + 8 + 4 * a, fl ? fl + 8 + 4 * a : NULL, 4, u24(d1.v[a]), have,
                                     (gp >> (4 + 2 * a)) & 3u, &lp_r[a]);
            q->roles[a] = (uint8_t)r;
            roles |= r << (2 * a);
        }
        q->topo = (uint8_t)topo; q->cnt = (uint8_t)cnt;
        q->keff = (uint8_t)keff_of(topo, cnt + 1);
        q->n_stages = (uint8_t)n_stages_of(topo, q->keff);
        q->stage = 0; q->pending = 0; q->succ = 0; q->planned = 1;
        float lp = lp_t + lp_c;
        for (uint32_t a = 0; a < q->keff; a++) lp = lp + lp_r[a];
        odec_t rec = {t, (uint16_t)qi, 0, 0, topo | (cnt << 2) | (roles << 4), lp, 0.0f};
        push_dec(&E->plan_log, &E->plan_logits, &E->n_plan, &E->cap_plan, 24, (int)s->keep_logits, rec, logits);
        E->ctr[C_PLANS]++;
    }

    /* ---- D EXEC (R15, R18, R24): queries with pending==0 and stages left, index ascending */
    for (uint32_t qi = 0; qi < s->qcap; qi++) {
        oq_t *q = &E->q[qi];
        if (!q->live || q->pending != 0 || q->stage >= q->n_stages) continue;
        uint32_t a0, nc;
        stage_calls(q->topo, q->keff, q->stage, &a0, &nc);
        for (uint32_t j = 0; j < nc; j++) {
            uint32_t agent = a0 + j;
            float b = (float)(q->deadline - t) / (float)s->budget_norm_ticks;
            if (b < -1.0f) b = -1.0f;
            if (b > 1.0f) b = 1.0f;
            shared_block(c, snap, b, q->in_tok, x);
            x[3 * N + 2 + q->topo] = 1.0f;
            x[3 * N + 6 + q->roles[agent]] = 1.0f;
            x[3 * N + 10] = (float)agent * 0.25f;
            x[3 * N + 11] = (float)q->keff * 0.25f;
            mlp_forward(c, &c->exec, x, logits);
            ph4 d = draw(c, STREAM_EXEC, gid, t, qi * 4u + agent, 0);
            const float *fl = NULL; int have = 0; uint32_t ga = 0;
            if (F && F->exec.off) {
                size_t cur = (size_t)F->exec.off[ei] + E->cur_exec;
                if (cur < (size_t)F->exec.off[ei + 1] && F->exec.t[cur] == t && F->exec.q[cur] == qi &&
                    F->exec.agent[cur] == agent) {
                    have = 1; ga = F->exec.payload[cur];
                    if (F->exec.logits) {
                        fl = F->exec.logits + cur * (3 * N + 1);
                        stat_logits(E, logits, fl, 3 * N);
                        double dv = fabs((double)logits[3 * N] - (double)fl[3 * N]);
                        if (!(dv <= E->max_value_diff)) E->max_value_diff = dv;
                    }
                    E->cur_exec++;
                } else E->n_desync++;
            }
            float lp;
            uint32_t a = decide_head(E, logits, fl, 3 * N, u24(d.v[0]), have, ga, &lp);
            uint32_t model = a / 3u, depth = a % 3u;
            odec_t rec = {t, (uint16_t)qi, (uint8_t)agent, 0, a, lp, fl ? fl[3 * N] : logits[3 * N]};
            push_dec(&E->exec_log, &E->exec_logits, &E->n_exec, &E->cap_exec, 3 * N + 1, (int)s->keep_logits, rec, logits);
            E->ctr[C_EXEC_DEC]++;
            /* R18 call issue */
            uint64_t prod = (uint64_t)s->depth_median_tok[depth] * c->tab_mult[d.v[1] >> 22];
            uint32_t out_total = (uint32_t)(prod >> 16);
            if (out_total < 1) out_total = 1;
            uint32_t ri = qi * 4u + agent;             /* R10: the call (query, agent) */
            or_t *r = &E->r[ri];
            r->state = ST_WAIT; r->slot = 0; r->model = (uint8_t)model; r->depth = (uint8_t)depth; r->agent = (uint8_t)agent;
            r->succ = d.v[2] < s->model[model].succ_thresh[depth];
            r->query = (uint16_t)qi; r->deadline = q->deadline; r->issue = t;
            r->remaining = out_total; r->out_total = out_total; r->prefill_us = 0; r->in_tok = q->in_tok;
            E->m[model].n_wait++;
            q->pending++;
            E->ctr[C_ISSUED]++;
        }
        q->stage++;
    }

    /* ---- E ADMIT (R20, R21): per model, WAITING in key order; stop at the first that does not fit */
    for (uint32_t k = 0; k < N; k++) {
        om_t *m = &E->m[k];
        for (;;) {
            if (m->n_wait == 0) break;
            int found = 0; uint32_t bi = 0;
            for (uint32_t i = 0; i < n_req(c); i++) {
                const or_t *r = &E->r[i];
                if (r->state != ST_WAIT || r->model != k) continue;
                if (!found || key_less(c, r, i, &E->r[bi], bi)) { found = 1; bi = i; }
            }
            or_t *r = &E->r[bi];
            uint32_t need = r->in_tok + (r->out_total - r->remaining);  /* R12 */
            if (!(m->n_run < s->model[k].slots && m->kv_used + need <= s->model[k].kv_cap)) break;
            r->slot = (uint8_t)lowest_free_slot(c, E, k);      /* R10 (n_run < slots, so one is free) */
            r->state = ST_RUN;
            r->prefill_us = (uint32_t)(((uint64_t)s->model[k].prefill_us_per_ktok * need) / 1000u);
            m->kv_used += need; m->n_wait--; m->n_run++;
        }
    }

    /* ---- F SERVE (R11): token-level service with stochastic rounding */
    for (uint32_t i = 0; i < n_req(c); i++) {
        or_t *r = &E->r[i];
        if (r->state != ST_RUN) continue;
        uint32_t usable = ORC_DT_US;
        uint32_t d = r->prefill_us < usable ? r->prefill_us : usable;
        r->prefill_us -= d; usable -= d;
        uint32_t xx = s->model[r->model].rate_tok_s * usable;
        uint32_t base = xx / 1000000u, frac = xx % 1000000u;
        /* R2/R11: sixteen-bit uniform of the request's slot; Bernoulli(frac) to 2^-16 */
        uint32_t gs = global_slot(c, r->model, r->slot), f = gs & 7u;
        uint32_t u16 = (draw(c, STREAM_SVC, gid, t, gs >> 3, 0).v[f >> 1] >> (16u * (f & 1u))) & 0xFFFFu;
        uint32_t thr = (uint32_t)(((uint64_t)frac << 16) / 1000000u);
        uint32_t extra = u16 < thr ? 1u : 0u;
        uint32_t tok = base + extra;
        if (tok > r->remaining) tok = r->remaining;
        r->remaining -= tok;
        E->m[r->model].kv_used += tok;
    }

    /* ---- G COMPLETE (R1, R13, R27, R28) */
    uint32_t lat_sum[ORC_MAXN] = {0}, lat_n[ORC_MAXN] = {0};
    for (uint32_t i = 0; i < n_req(c); i++) {
        or_t *r = &E->r[i];
        if (r->state != ST_RUN || r->remaining != 0) continue;
        oq_t *q = &E->q[r->query];
        uint32_t ell = (uint32_t)(t + 1 - r->issue);
        lat_sum[r->model] += ell; lat_n[r->model]++;
        cost_q16 += ((uint64_t)ell << 16) / q->budget;     /* C_k = l_k / beta */
        q->succ |= r->succ;                                /* R19 */
        q->pending--;
        E->m[r->model].kv_used -= r->in_tok + r->out_total;
        E->m[r->model].n_run--;
        E->ctr[C_CALLS_DONE]++;
        memset(r, 0, sizeof(*r));
    }
    for (uint32_t k = 0; k < N; k++) {
        if (lat_n[k] == 0) continue;
        int32_t mean_q8 = (int32_t)((lat_sum[k] << 8) / lat_n[k]);
        int32_t ew = (int32_t)E->m[k].ewma_q8;
        ew += (mean_q8 - ew) >> 3;                         /* R13: alpha = 1/8, arithmetic shift */
        E->m[k].ewma_q8 = (uint32_t)ew;
    }
    for (uint32_t qi = 0; qi < s->qcap; qi++) {
        oq_t *q = &E->q[qi];
        if (!q->live || q->pending != 0 || q->stage < q->n_stages) continue;
        uint32_t sojourn = (uint32_t)(t + 1 - q->arrive);
        uint32_t late = (t + 1 > q->deadline) ? 1u : 0u;
        rew += q->succ; miss += late;
        E->ctr[C_FINISHED]++; E->ctr[C_SOLVED] += q->succ; E->ctr[C_MISSED] += late; E->ctr[C_SUM_SOJOURN] += sojourn;
        if (E->n_qlog == E->cap_qlog) {
            E->cap_qlog = E->cap_qlog ? E->cap_qlog * 2 : 64;
            E->qlog = (oqlog_t *)realloc(E->qlog, E->cap_qlog * sizeof(oqlog_t));
        }
        oqlog_t ql = {gid, q->budget | ((uint32_t)q->succ << 16) | ((uint32_t)q->topo << 17) | ((uint32_t)q->keff << 19), q->arrive, sojourn};
        E->qlog[E->n_qlog++] = ql;
        memset(q, 0, sizeof(*q));
    }

    /* ---- H PREEMPT (R21): evict the RUNNING request with the largest (deadline, ridx) */
    if (s->kv_preempt) {
        for (uint32_t k = 0; k < N; k++) {
            om_t *m = &E->m[k];
            while (m->kv_used > s->model[k].kv_cap) {
                int found = 0; uint32_t vi = 0; int32_t vd = 0;
                for (uint32_t i = 0; i < n_req(c); i++) {
                    const or_t *r = &E->r[i];
                    if (r->state != ST_RUN || r->model != k) continue;
                    if (!found || r->deadline > vd || (r->deadline == vd && i > vi)) { found = 1; vd = r->deadline; vi = i; }
                }
                if (!found) break;
                or_t *r = &E->r[vi];
                m->kv_used -= r->in_tok + (r->out_total - r->remaining);
                r->state = ST_WAIT; r->prefill_us = 0; r->slot = 0;
                m->n_run--; m->n_wait++;
                E->ctr[C_PREEMPT]++;
            }
        }
    }

    /* ---- I RECORD (R27, R28, R33) */
    size_t idx = (size_t)trow * c->n_envs + ei;
    c->rew[idx] = (float)rew;
    c->cost[idx] = s->cost_mode ? (float)miss : (float)cost_q16 * 0x1p-16f;
    c->miss[idx] = (uint8_t)(miss > 255 ? 255 : miss);
    uint32_t done = (s->episode_ticks && ((uint32_t)(t + 1) % s->episode_ticks) == 0) ? 1u : 0u;
    c->done[idx] = (uint8_t)done;
    for (uint32_t k = 0; k < N; k++) { E->ctr[C_SUM_RUNNING] += E->m[k].n_run; E->ctr[C_SUM_WAITING] += E->m[k].n_wait; }
    if (done) {                                            /* hard reset, live queries abandoned */
        for (uint32_t i = 0; i < s->qcap; i++) E->ctr[C_ABANDONED] += E->q[i].live;
        memset(E->q, 0, sizeof(oq_t) * s->qcap);
        memset(E->r, 0, sizeof(or_t) * n_req(c));
        memset(E->m, 0, sizeof(E->m));
    }
}

/* --------------------------------------------------------------------------------------- API */
int orc_create(const orc_spec *spec, uint32_t n_envs, const uint32_t *env_ids, const uint8_t *env_level,
               uint64_t seed, orc_ctx **out)
{
    if (!spec || !out || !n_envs || !env_ids || !env_level) return -1;
    if (spec->n_models == 0 || spec->n_models > ORC_MAXN || spec->rcap < 3 * spec->qcap || spec->rcap > 4096 || spec->qcap > 1024 ||
        spec->f_in > 512 || spec->hidden > 512 || spec->f_in < 3 * spec->n_models + 12) return -2;
    orc_ctx *c = (orc_ctx *)calloc(1, sizeof(orc_ctx));
    c->s = *spec;
    c->n_envs = n_envs; c->seed = seed;
    c->env_id = (uint32_t *)malloc(4 * n_envs); memcpy(c->env_id, env_ids, 4 * n_envs);
    c->env_level = (uint8_t *)malloc(n_envs); memcpy(c->env_level, env_level, n_envs);
    c->tab_mult = (uint32_t *)malloc(4096); memcpy(c->tab_mult, spec->out_tok_mult_q16, 4096);
    if (spec->in_tok_table) { c->tab_intok = (uint32_t *)malloc(4096); memcpy(c->tab_intok, spec->in_tok_table, 4096); }
    c->tab_cdf = (uint32_t *)malloc(128u * spec->n_levels); memcpy(c->tab_cdf, spec->arr_cdf, 128u * spec->n_levels);
    c->s.out_tok_mult_q16 = c->s.in_tok_table = c->s.arr_cdf = NULL;
    c->env = (oenv_t *)calloc(n_envs, sizeof(oenv_t));
    for (uint32_t i = 0; i < n_envs; i++) {
        c->env[i].q = (oq_t *)calloc(spec->qcap, sizeof(oq_t));
        c->env[i].r = (or_t *)calloc(4u * spec->qcap, sizeof(or_t));
    }
    size_t rows = (size_t)spec->max_ticks + 1;
    c->rew = (float *)calloc(rows * n_envs, 4); c->cost = (float *)calloc(rows * n_envs, 4);
    c->val = (float *)calloc(rows * n_envs, 4);
    c->done = (uint8_t *)calloc(rows * n_envs, 1); c->miss = (uint8_t *)calloc(rows * n_envs, 1);
    c->adv = (double *)calloc(rows * n_envs, 8); c->ret = (double *)calloc(rows * n_envs, 8);
    *out = c;
    return 0;
}

static void clear_logs(orc_ctx *c)
{
    for (uint32_t i = 0; i < c->n_envs; i++) {
        oenv_t *E = &c->env[i];
        E->n_plan = E->n_exec = E->n_qlog = 0;
        E->cur_plan = E->cur_exec = 0;
    }
}

int orc_reset(orc_ctx *c)
{
    if (!c) return -1;
    for (uint32_t i = 0; i < c->n_envs; i++) {
        oenv_t *E = &c->env[i];
        memset(E->q, 0, sizeof(oq_t) * c->s.qcap);
        memset(E->r, 0, sizeof(or_t) * n_req(c));
        memset(E->m, 0, sizeof(E->m));
        memset(E->ctr, 0, sizeof(E->ctr));
        E->n_desync = E->n_hard = E->n_near = 0; E->max_logit_diff = E->max_value_diff = 0.0;
    }
    clear_logs(c);
    c->tick = 0; c->last_T = 0; c->have_returns = 0;
    return 0;
}

void orc_destroy(orc_ctx *c)
{
    if (!c) return;
    for (uint32_t i = 0; i < c->n_envs; i++) {
        oenv_t *E = &c->env[i];
        free(E->q); free(E->r); free(E->plan_log); free(E->exec_log); free(E->plan_logits); free(E->exec_logits); free(E->qlog);
    }
    free(c->env); free(c->env_id); free(c->env_level); free(c->tab_mult); free(c->tab_intok); free(c->tab_cdf);
    free(c->rew); free(c->cost); free(c->val); free(c->done); free(c->miss); free(c->adv); free(c->ret); free(c->wbuf);
    free(c);
}

int orc_set_forced(orc_ctx *c, const orc_forced *f) { c->forced = f; return 0; }

/* advance every env by n_ticks; trajectory rows 0..n_ticks-1, row n_ticks of val = bootstrap (R30) */
int orc_rollout(orc_ctx *c, const void *blob, uint32_t n_ticks, int n_threads)
{
    if (!c || !blob) return -1;
    if (n_ticks > c->s.max_ticks) return -6;
    int rc = load_blob(c, (const uint8_t *)blob);
    if (rc) return rc;
    clear_logs(c);
    const int32_t t0 = c->tick;
    const uint32_t N = c->s.n_models;
#ifdef _OPENMP
    if (n_threads < 1) n_threads = 1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads)
#endif
    for (uint32_t ei = 0; ei < c->n_envs; ei++) {
        for (uint32_t k = 0; k < n_ticks; k++) env_tick(c, ei, t0 + (int32_t)k, k);
        float x[512], logits[64];
        shared_block(c, c->env[ei].m, 0.0f, 0, x);
        mlp_forward(c, &c->exec, x, logits);
        c->val[(size_t)n_ticks * c->n_envs + ei] = logits[3 * N];
    }
    (void)n_threads;
    c->tick = t0 + (int32_t)n_ticks;
    c->last_T = n_ticks;
    c->have_returns = 0;
    return 0;
}

/* R31 GAE (float64 recurrence on the float32 trajectory) with the Lagrangian reward R29:
 * r~ = rew - mu*cost; delta = r~ + (nd ? gamma*V[t+1] : 0) - V[t]; A[t] = delta + (nd ? gamma*lam*A[t+1] : 0);
 * ret[t] = A[t] + V[t]; A[T] = 0.  Standalone so that bf16 parity can feed it the GPU's arrays. */
int orc_gae(const float *rew, const float *cost, const float *val, const uint8_t *done, uint32_t T, uint32_t n,
            double gamma, double lam, double mu, double *adv, double *ret)
{
    for (uint32_t e = 0; e < n; e++) {
        double A = 0.0;
        for (int64_t t = (int64_t)T - 1; t >= 0; t--) {
            size_t i = (size_t)t * n + e;
            int nd = !done[i];
            double rt = (double)rew[i] - mu * (double)cost[i];
            double delta = rt + (nd ? gamma * (double)val[i + n] : 0.0) - (double)val[i];
            A = delta + (nd ? gamma * lam * A : 0.0);
            adv[i] = A;
            ret[i] = A + (double)val[i];
        }
    }
    return 0;
}

/* im_returns: GAE (a), planner utility U_i and its normalisation (b, R32), C-bar (c) */
int orc_returns(orc_ctx *c, double gamma, double lam, double mu)
{
    if (!c) return -1;
    if (c->last_T == 0) return -5;
    orc_gae(c->rew, c->cost, c->val, c->done, c->last_T, c->n_envs, gamma, lam, mu, c->adv, c->ret);
    double sc = 0.0;
    for (size_t i = 0; i < (size_t)c->last_T * c->n_envs; i++) sc += (double)c->cost[i];
    uint64_t nf = 0; double su = 0.0, su2 = 0.0;
    for (uint32_t e = 0; e < c->n_envs; e++)
        for (size_t j = 0; j < c->env[e].n_qlog; j++) {
            const oqlog_t *q = &c->env[e].qlog[j];
            double U = (double)((q->info >> 16) & 1u) - mu * (double)q->sojourn / (double)(q->info & 0xFFFFu);
            su += U; su2 += U * U; nf++;
        }
    c->sum_cost = sc; c->n_final = nf;
    c->cbar = nf ? sc / (double)nf : 0.0;
    c->ubar = nf ? su / (double)nf : 0.0;
    double var = nf ? su2 / (double)nf - c->ubar * c->ubar : 0.0;
    c->usigma = sqrt(var > 0.0 ? var : 0.0);
    c->have_returns = 1;
    return 0;
}

/* ------------------------------------------------------------------------------------ read-out */
enum { ORC_REW = 1, ORC_COST, ORC_VAL, ORC_DONE, ORC_MISS, ORC_ADV, ORC_RET, ORC_COUNTERS, ORC_SNAPSHOT, ORC_STATE,
       ORC_SCALARS, ORC_STATS };

size_t orc_state_words(const orc_ctx *c) { return 4u * c->s.n_models + 4u * c->s.qcap + 5u * 4u * c->s.qcap; }

static void dump_state(const orc_ctx *c, const oenv_t *E, uint32_t *w)
{
    for (uint32_t k = 0; k < c->s.n_models; k++) {
        *w++ = E->m[k].n_wait; *w++ = E->m[k].n_run; *w++ = E->m[k].kv_used; *w++ = E->m[k].ewma_q8;
    }
    for (uint32_t i = 0; i < c->s.qcap; i++) {
        const oq_t *q = &E->q[i];
        if (!q->live) { w[0] = w[1] = w[2] = w[3] = 0; w += 4; continue; }
        uint32_t roles = q->roles[0] | (q->roles[1] << 2) | (q->roles[2] << 4) | (q->roles[3] << 6);
        *w++ = 1u | ((uint32_t)q->planned << 1) | ((uint32_t)q->topo << 2) | ((uint32_t)q->cnt << 4) | ((uint32_t)q->keff << 6) |
               ((uint32_t)q->stage << 9) | ((uint32_t)q->n_stages << 12) | ((uint32_t)q->pending << 15) |
               ((uint32_t)q->succ << 17) | (roles << 18);
        *w++ = (uint32_t)q->deadline; *w++ = (uint32_t)q->arrive; *w++ = q->budget | (q->in_tok << 16);
    }
    for (uint32_t i = 0; i < n_req(c); i++) {
        const or_t *r = &E->r[i];
        if (r->state == ST_FREE) { w[0] = w[1] = w[2] = w[3] = w[4] = 0; w += 5; continue; }
        *w++ = r->state | ((uint32_t)r->model << 2) | ((uint32_t)r->depth << 6) | ((uint32_t)r->agent << 8) |
               ((uint32_t)r->succ << 10) | ((uint32_t)r->query << 16);
        *w++ = (uint32_t)r->deadline; *w++ = (uint32_t)r->issue;
        /* prefill is sub-tick (R11), hence 0 at every tick boundary; the field carries slot+1 of a RUNNING request */
        *w++ = r->remaining | ((r->state == ST_RUN ? (uint32_t)r->slot + 1u : 0u) << 16); *w++ = r->out_total | (r->in_tok << 16);
    }
}

/* copies `what` into dst (caller-sized); returns bytes written or <0 */
int64_t orc_read(orc_ctx *c, uint32_t what, void *dst, size_t cap)
{
    size_t n = c->n_envs, T = c->last_T, bytes = 0;
    const void *src = NULL;
    switch (what) {
    case ORC_REW: src = c->rew; bytes = 4 * T * n; break;
    case ORC_COST: src = c->cost; bytes = 4 * T * n; break;
    case ORC_VAL: src = c->val; bytes = 4 * (T + 1) * n; break;
    case ORC_DONE: src = c->done; bytes = T * n; break;
    case ORC_MISS: src = c->miss; bytes = T * n; break;
    case ORC_ADV: if (!c->have_returns) return -5; src = c->adv; bytes = 8 * T * n; break;
    case ORC_RET: if (!c->have_returns) return -5; src = c->ret; bytes = 8 * T * n; break;
    case ORC_COUNTERS: {
        bytes = 8 * C_N * n; if (cap < bytes) return -6;
        for (size_t e = 0; e < n; e++) memcpy((uint64_t *)dst + e * C_N, c->env[e].ctr, 8 * C_N);
        return (int64_t)bytes; }
    case ORC_SNAPSHOT: {
        bytes = 16 * c->s.n_models * n; if (cap < bytes) return -6;
        for (size_t e = 0; e < n; e++) memcpy((uint32_t *)dst + e * 4 * c->s.n_models, c->env[e].m, 16 * c->s.n_models);
        return (int64_t)bytes; }
    case ORC_STATE: {
        bytes = 4 * orc_state_words(c) * n; if (cap < bytes) return -6;
        for (size_t e = 0; e < n; e++) dump_state(c, &c->env[e], (uint32_t *)dst + e * orc_state_words(c));
        return (int64_t)bytes; }
    case ORC_SCALARS: {
        if (!c->have_returns) return -5;
        bytes = 8 * 5; if (cap < bytes) return -6;
        double v[5] = {c->cbar, c->ubar, c->usigma, c->sum_cost, (double)c->n_final};
        memcpy(dst, v, bytes); return (int64_t)bytes; }
    case ORC_STATS: {
        bytes = 8 * 5; if (cap < bytes) return -6;
        double v[5] = {0, 0, 0, 0, 0};
        for (size_t e = 0; e < n; e++) {
            v[0] += (double)c->env[e].n_desync; v[1] += (double)c->env[e].n_hard; v[2] += (double)c->env[e].n_near;
            if (!(c->env[e].max_logit_diff <= v[3])) v[3] = c->env[e].max_logit_diff;
            if (!(c->env[e].max_value_diff <= v[4])) v[4] = c->env[e].max_value_diff;
        }
        memcpy(dst, v, bytes); return (int64_t)bytes; }
    default: return -1;
    }
    if (cap < bytes) return -6;
    memcpy(dst, src, bytes);
    return (int64_t)bytes;
}

/* decision / query logs, env-major then chronological */
int64_t orc_log_count(const orc_ctx *c, int kind)
{
    size_t n = 0;
    for (uint32_t e = 0; e < c->n_envs; e++) n += kind == 0 ? c->env[e].n_plan : kind == 1 ? c->env[e].n_exec : c->env[e].n_qlog;
    return (int64_t)n;
}

int orc_read_decisions(const orc_ctx *c, int kind, uint32_t *env_local, int32_t *t, uint16_t *q, uint8_t *agent,
                       uint32_t *payload, float *logp, float *value, float *logits)
{
    size_t k = 0;
    const uint32_t n_out = kind ? 3 * c->s.n_models + 1 : 24;
    for (uint32_t e = 0; e < c->n_envs; e++) {
        const oenv_t *E = &c->env[e];
        const odec_t *log = kind ? E->exec_log : E->plan_log;
        const float *lg = kind ? E->exec_logits : E->plan_logits;
        size_t n = kind ? E->n_exec : E->n_plan;
        for (size_t j = 0; j < n; j++, k++) {
            env_local[k] = e; t[k] = log[j].t; q[k] = log[j].q; agent[k] = log[j].agent;
            payload[k] = log[j].payload; logp[k] = log[j].logp; value[k] = log[j].value;
            if (logits && c->s.keep_logits) memcpy(logits + k * n_out, lg + j * n_out, 4 * n_out);
        }
    }
    return 0;
}

int orc_read_queries(const orc_ctx *c, uint32_t *env, int32_t *arrive, uint32_t *sojourn, uint32_t *info)
{
    size_t k = 0;
    for (uint32_t e = 0; e < c->n_envs; e++)
        for (size_t j = 0; j < c->env[e].n_qlog; j++, k++) {
            const oqlog_t *r = &c->env[e].qlog[j];
            env[k] = r->env; arrive[k] = r->arrive; sojourn[k] = r->sojourn; info[k] = r->info;
        }
    return 0;
}

/* R20/R21 helper for the P9 pin and QUEUE_ORDER parity: WAITING requests of env `ei`, model k, in key order at tick t */
int orc_queue_order(const orc_ctx *c, uint32_t ei, uint32_t k, int32_t t, uint32_t *ridx_out, uint32_t cap)
{
    const oenv_t *E = &c->env[ei];
    uint32_t n = 0, last = 0;
    int have_last = 0;
    (void)t;                 /* the order at a fixed t does not depend on t (R20) */
    for (;;) {
        uint32_t bi = 0; int found = 0;
        for (uint32_t i = 0; i < n_req(c); i++) {
            const or_t *r = &E->r[i];
            if (r->state != ST_WAIT || r->model != k) continue;
            if (have_last && !key_less(c, &E->r[last], last, r, i)) continue;   /* only those after `last` */
            if (!found || key_less(c, r, i, &E->r[bi], bi)) { bi = i; found = 1; }
        }
        if (!found) break;
        if (n < cap) ridx_out[n] = bi;
        n++; last = bi; have_last = 1;
    }
    return (int)n;
}

int32_t orc_tick(const orc_ctx *c) { return c->tick; }
