/*
 * inframind.h — C ABI of libinframind.so: B200-native (sm_100a) rollout of the INFRAMIND hierarchical
 * constrained MDP over many independent simulated LLM-server pools, plus GAE / Lagrangian returns.
 *
 * Source of each call: BASELINE.json `north_star` names the five calls im_create / im_reset / im_rollout /
 * im_returns / im_read_telemetry; SURVEY.md §8(b) adds the minimum auxiliaries (arena binding, errors).
 * The operations themselves follow the paper's problem statement (pool of N services,
 * queries with budget beta, planner + executor policies, Lagrangian objective) and the numbered Readings
 * R1..R34 in DESIGN.md.
 *
 * Conventions
 *   - Every call returns an int: IM_OK or a negative im_status. No C++ exception crosses the ABI.
 *   - No global state; one ctx is not thread-safe, separate ctxs are independent.
 *   - "host" / "device" is stated for every pointer. The library never allocates device memory itself:
 *     the caller lends ONE device arena (im_bind), e.g. a torch.uint8 tensor, plus the CUDA stream all
 *     work is enqueued on.
 *   - There is NO CPU fallback: without a CUDA device of compute capability 10.x every compute call fails
 *     with IM_ERR_CUDA (north_star: "no multi-backend dispatch and no CPU fallback").
 */
#ifndef INFRAMIND_H
#define INFRAMIND_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define IM_ABI_VERSION 1u
#define IM_MAX_MODELS 16u
#define IM_DT_US 50000u              /* one tick = 50 ms (north_star) */

typedef enum im_status {
    IM_OK = 0,
    IM_ERR_INVALID_ARG = -1,         /* null / zero / misaligned argument */
    IM_ERR_BAD_SPEC = -2,            /* N>16, RCAP<3*QCAP, non-monotone CDF row, zero slots, unsupported MLP shape ... */
    IM_ERR_CUDA = -3,                /* CUDA runtime error or no sm_100 device */
    IM_ERR_NOMEM = -4,               /* arena too small / host allocation failed */
    IM_ERR_STATE = -5,               /* call out of order (returns before rollout, read of ADV before returns, not bound) */
    IM_ERR_CAPACITY = -6             /* n_ticks > max_ticks, dst too small (*written = needed size), log overflow */
} im_status;

/* spec.debug_flags */
#define IM_FLAG_LOG_DECISIONS 1u     /* keep every planner / executor decision of the rollout (needed by a PPO step) */
#define IM_FLAG_LOG_LOGITS 2u        /* additionally keep the fp32 logits of every decision (parity tests, R25) */

/* spec.sched_mode (PAPER.md:117-119 EDF; FCFS is the paper's ablation) */
#define IM_SCHED_FCFS 0u
#define IM_SCHED_EDF 1u

/* spec.policy_dtype */
#define IM_DTYPE_F32 0u              /* R22: k-ascending FFMA, bit-exact against the oracle */
#define IM_DTYPE_BF16 1u             /* R25: bf16 operands, fp32 accumulation, tensor cores */

typedef struct im_model_spec {
    uint32_t rate_tok_s;             /* decode tokens/s per RUNNING request (R11) */
    uint32_t slots;                  /* S_k concurrent requests (PAPER.md:275 max_num_seqs) */
    uint32_t kv_cap;                 /* KV capacity in tokens (R12) */
    uint32_t prefill_us_per_ktok;    /* prefill microseconds per 1000 input tokens (R11) */
    uint32_t succ_thresh[3];         /* floor(p[k][depth] * 2^32): call succeeds iff u32 draw < thresh (R18) */
    float kv_inv;                    /* fp32(1/kv_cap): d_kv feature scale (R14) */
} im_model_spec;

/* Plain-old-data description of pool + workload. All dynamics parameters are integers (R4).
 * Ownership: the four table pointers are HOST pointers; im_create deep-copies everything, the caller may
 * free them immediately afterwards. */
typedef struct im_pool_spec {
    uint32_t abi_version;            /* IM_ABI_VERSION */
    uint32_t n_models;               /* N <= 16 */
    uint32_t qcap;                   /* query-table slots per env, multiple of 32, <= 1024 (R9) */
    uint32_t rcap;                   /* waiting-list capacity per env, multiple of 128, >= 3*qcap, <= 4096: a query has at most
                                        3 calls in flight (R17), so the list never overflows (R9) */
    uint32_t max_ticks;              /* trajectory capacity of one im_rollout, <= 8191 */
    uint32_t sched_mode;             /* IM_SCHED_* (R20) */
    uint32_t kv_preempt;             /* 1: evict when kv_used > kv_cap (R21) */
    uint32_t cost_mode;              /* 0: cost = sum l/beta; 1: cost = SLO-miss count (R28) */
    uint32_t episode_ticks;          /* 0: continuing; >0: done + hard reset every episode_ticks ticks (R33) */
    uint32_t budget_norm_ticks;      /* budget feature normaliser (R15) */
    uint32_t n_levels;               /* arrival-rate levels, <= 256 (R6) */
    uint32_t policy_dtype;           /* IM_DTYPE_* */
    uint32_t f_in;                   /* MLP input width >= 3N+12 (R15); fp32: multiple of 4 <= 128; bf16: 64 or 128 */
    uint32_t hidden;                 /* MLP hidden width; fp32: multiple of 32 <= 256; bf16: 128 or 256 */
    uint32_t debug_flags;            /* IM_FLAG_* */
    uint32_t in_tok_const;           /* input tokens per query when in_tok_table == NULL (R8) */
    uint32_t mix_thresh;             /* budget mixture: component 0 iff u32 draw < mix_thresh (R7) */
    uint32_t env_id_base;            /* global id of env 0: Philox keys use env_id_base + e (R2; multi-GPU shards) */
    uint32_t depth_median_tok[3];    /* output-token medians per depth (R18) */
    uint32_t mix_lo[2], mix_hi[2];   /* budget components, ticks, inclusive (R7); hi <= 65535 */
    uint32_t reserved;
    uint64_t log_cap_exec;           /* rows of the executor decision log of one im_rollout (0 = default); used only with
                                        IM_FLAG_LOG_DECISIONS: without it the work list is a ring sized by the library */
    uint64_t log_cap_plan;           /* the same for the planner */
    uint64_t log_cap_query;          /* capacity (records) of the finished-query log */
    im_model_spec model[IM_MAX_MODELS];
    const uint32_t *out_tok_mult_q16;/* HOST [1024]: Q16 output-token multipliers (lognormal quantiles, R18) */
    const uint32_t *in_tok_table;    /* HOST [1024] or NULL: input-token quantile table (R8) */
    const uint32_t *arr_cdf;         /* HOST [n_levels][32]: Poisson thresholds floor(F(j)*2^32), j<31 used (R5) */
    const uint8_t *env_level;        /* HOST [n_envs]: arrival level of each env (R6) */
} im_pool_spec;

typedef struct im_ctx im_ctx;        /* opaque, owned by the library */

/* Bytes of device arena needed for (spec, n_envs); 0 if the spec is invalid. Host-only computation. */
size_t im_arena_bytes(const im_pool_spec *spec, uint32_t n_envs);

/* Validate + deep-copy the spec (host). `seed` keys every Philox stream (R2). No device work happens here. */
int im_create(const im_pool_spec *spec, uint32_t n_envs, uint64_t seed, im_ctx **out);

/* Lend the device arena (DEVICE pointer, 256-byte aligned, >= im_arena_bytes) and the CUDA stream
 * (cudaStream_t as void*, NULL = default stream). Uploads the tables and resets the state (as im_reset).
 * The arena must stay alive and untouched by the caller until im_destroy. */
int im_bind(im_ctx *ctx, void *dev_arena, size_t bytes, void *cuda_stream);

/* Empty pools, tick = 0, counters = 0. The same seed then replays identically (P15). Asynchronous. */
int im_reset(im_ctx *ctx);

/* Advance every env by n_ticks <= max_ticks fixed 50 ms ticks under the given policy (canonical tick
 * A..I of DESIGN.md).  `policy_weights` is the R26 blob, HOST or DEVICE pointer (detected; a host blob is
 * checked and copied before the call returns, pinned or not; a device blob must stay valid until the stream has
 * passed the call, and a header that does not match the spec surfaces as IM_ERR_BAD_SPEC at the next
 * im_read_telemetry).  Overwrites trajectory rows 0..n_ticks-1 (row n_ticks of VAL = bootstrap
 * value) and the decision / query logs.  Env state persists across calls (split-invariance, P15).
 * Asynchronous on the bound stream. */
int im_rollout(im_ctx *ctx, const void *policy_weights, uint32_t n_ticks);

/* Over the last rollout: (a) GAE with Lagrangian reward r - mu*cost (Eq. 3; R29, R31) -> ADV, RET;
 * (b) planner utility U_i = solved - mu*L_total/beta, normalised by batch mean/std (Eq. 6; R32);
 * (c) C-bar = sum(cost)/#finished for the dual update (Eq. 7). Asynchronous. */
int im_returns(im_ctx *ctx, float gamma, float lambda, float lagrange_mu);

/* Env-sharded jobs (one ctx per GPU): every rank calls im_returns, the four sums of IM_TEL_SUMS are
 * added over the ranks (the job's ONE collective, e.g. an NCCL all-reduce of 4 doubles), and every rank calls
 * im_returns_finish with the job-wide sums (HOST array of 4 doubles, same order as IM_TEL_SUMS).  UNORM is then
 * re-normalised with the job's U-bar / sigma_U (Eq. 6) and SCALARS reports the job's C-bar, U-bar,
 * sigma_U, sum_cost, n_finished: the sharded result equals the single-GPU result.  Without this call UNORM and
 * SCALARS are those of the ctx's own envs.  IM_ERR_STATE before im_returns.  Asynchronous. */
int im_returns_finish(im_ctx *ctx, const double *global_sums);

/* selectors of im_read_telemetry / im_device_ptr */
typedef enum im_telemetry {
    IM_TEL_SNAPSHOT = 1,   /* u32 [E][N][4] = {n_wait, n_run, kv_used, ewma_q8}: the paper's d vectors */
    IM_TEL_COUNTERS = 2,   /* u64 [E][16]: arrivals, dropped, finished, solved, missed, calls_issued, calls_done,
                              preemptions, sum_sojourn, sum_live_mid, plans, exec_decisions, sum_running,
                              sum_waiting, near_boundary(=0), abandoned */
    IM_TEL_REW = 3,        /* f32 [T][E] */
    IM_TEL_COST = 4,       /* f32 [T][E] */
    IM_TEL_VAL = 5,        /* f32 [T+1][E] */
    IM_TEL_DONE = 6,       /* u8  [T][E] */
    IM_TEL_MISS = 7,       /* u8  [T][E] (saturating) */
    IM_TEL_ADV = 8,        /* f32 [T][E]   (after im_returns) */
    IM_TEL_RET = 9,        /* f32 [T][E]   (after im_returns) */
    IM_TEL_SCALARS = 10,   /* f64 [8]: cbar, ubar, usigma, sum_cost, n_finished (of the ctx, or of the job after
                              im_returns_finish), n_exec_decisions, n_plan_decisions, tick */
    IM_TEL_DECISIONS_EXEC = 11, /* u32 [n][6]: env(global), t(abs), q | agent<<16, action, logp(f32 bits), value(f32 bits) */
    IM_TEL_DECISIONS_PLAN = 12, /* u32 [n][6]: env(global), t(abs), q, topo | cnt<<2 | roles<<4, logp(f32 bits), 0 */
    IM_TEL_QUERIES = 13,   /* u32 [n][4]: env(global), arrive, sojourn, budget | solved<<16 | topo<<17 | keff<<19 */
    IM_TEL_UNORM = 14,     /* f32 [n]: normalised utility of each QUERIES record, same order (after im_returns) */
    IM_TEL_STATE = 15,     /* u32 [E][4N + 4*QCAP + 5*(4*QCAP)]: canonical full state dump, layout below */
    IM_TEL_QUEUE_ORDER = 16,/* u32 [E][N+1 + RCAP]: per env N+1 segment offsets, then the WAITING request ids (4*query + agent)
                              of model 0, model 1, ... each in slack (R20 key) order; unused tail = 0xFFFFFFFF */
    IM_TEL_TABLES = 17,    /* u32: out_tok_mult_q16[1024], in_tok[1024], arr_cdf[n_levels*32] as uploaded */
    IM_TEL_LOGITS_EXEC = 18,/* f32 [n][3N+1], same order as DECISIONS_EXEC (needs IM_FLAG_LOG_LOGITS) */
    IM_TEL_LOGITS_PLAN = 19,/* f32 [n][24] */
    IM_TEL_SUMS = 20       /* f64 [4]: the raw sums of THIS ctx behind the scalars (after im_returns): sum of cost,
                              number of finalised queries, sum of U_i, sum of U_i^2 - what an env-sharded job
                              all-reduces before im_returns_finish */
} im_telemetry;

/* STATE dump, per env (free slots are all-zero words):
 *   model k : n_wait, n_run, kv_used, ewma_q8
 *   query i : w0 = live | planned<<1 | topo<<2 | (K-1)<<4 | keff<<6 | stage<<9 | n_stages<<12 | pending<<15 |
 *                  solved<<17 | roles(4x2b)<<18 ; w1 = deadline ; w2 = arrive ; w3 = budget | in_tok<<16
 *   request i = 4*query + agent (R10), i < 4*QCAP:
 *              w0 = state(0 free,1 waiting,2 running) | model<<2 | depth<<6 | agent<<8 | succ<<10 | query<<16 ;
 *              w1 = deadline ; w2 = issue ; w3 = remaining | (slot+1 if running else 0)<<16 ; w4 = out_total | in_tok<<16
 * Device-side limits: slots <= 64 per model, input / output tokens <= 8191 per call, absolute tick + largest budget
 * < 65536 (im_rollout returns IM_ERR_CAPACITY beyond; im_reset restarts the clock). */

/* Synchronise the stream and copy the selected telemetry to caller-owned HOST memory `dst`.
 * *written receives the byte count (or the needed size with IM_ERR_CAPACITY). dst == NULL queries the size. */
int im_read_telemetry(im_ctx *ctx, uint32_t what, void *dst, size_t dst_bytes, size_t *written);

/* DEVICE pointer + byte size of a trajectory array (REW, COST, VAL, DONE, MISS, ADV, RET) inside the arena,
 * for zero-copy consumers on the same stream (a PPO step). No synchronisation. */
int im_device_ptr(im_ctx *ctx, uint32_t what, void **dev_ptr, size_t *bytes);

/* Number of kernels this ctx has launched so far (bench.py's gpu_launches). */
uint64_t im_launch_count(const im_ctx *ctx);

/* Per-kernel-class device timing for roofline reports: when enabled, every launch of im_rollout / im_returns is
 * bracketed by CUDA events on the bound stream. im_kernel_times synchronises, returns the accumulated
 * milliseconds and launch counts per class since the last call, and clears them. HOST arrays of IM_KERNEL_CLASSES. */
#define IM_KERNEL_SIM 0       /* k_sim: tick phases A, B, D-issue, E, G .. I */
#define IM_KERNEL_PLAN 1      /* planner MLP + sampling */
#define IM_KERNEL_EXEC 2      /* executor + critic MLP + sampling */
#define IM_KERNEL_RETURNS 3   /* GAE + utility kernels of one im_returns */
#define IM_KERNEL_SERVE 4     /* k_serve: tick phase F (token-level service pass) */
#define IM_KERNEL_CLASSES 5
int im_set_profiling(im_ctx *ctx, int enable);
int im_kernel_times(im_ctx *ctx, double *ms, uint64_t *launches);

/* The returns kernel for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): GAE with the Lagrangian reward r - mu C (Eq. 3; R29, R31), the same arithmetic
 * as im_returns, on plain DEVICE arrays of the caller, without a ctx and without ANY allocation: the kernel's scratch
 * memory (one partial cost sum per 256 envs and a ticket) is a static device array of 33 024 bytes inside the library,
 * held by every GPU that loads the library until the process exits.
 *   rew, cost   [n_ticks][n_envs] f32 (env fastest)       val  [n_ticks + 1][n_envs] f32 (row n_ticks = bootstrap value, R30)
 *   done        [n_ticks][n_envs] u8 (R33)                adv, ret  [n_ticks][n_envs] f32, written
 *   sum_cost    one f64, written: sum of cost over all rows (numerator of C-bar, Eq. 7), added up in a
 *               fixed order (the same bits in every run); may be NULL
 *   cuda_stream cudaStream_t (may be NULL); asynchronous: the results are valid after the stream has synchronised
 *   errbuf      optional host buffer that receives the message of a failing call ("" on success)
 * All arrays are caller-owned; device pointers of the CURRENT device.  n_envs > IM_GAE_STATIC_MAX_ENVS is refused with
 * IM_ERR_CAPACITY (split the batch by env ranges, or use im_returns); null arrays or zero sizes IM_ERR_INVALID_ARG; a
 * CUDA failure IM_ERR_CUDA.  Calls no cudaMalloc / cudaFree or allocating routine; the first call on a device looks the
 * scratch address up (cudaGetSymbolAddress), so make one call per device before capturing a graph.
 * EVERY call on a device shares the one scratch array: calls that overlap on the GPU (different streams, or graphs
 * replayed concurrently) race on it and return a wrong sum_cost; calls ordered on one stream are safe (each call clears
 * the ticket it needs at zero; the partial sums are rewritten before they are read). */
#define IM_GAE_STATIC_MAX_ENVS 1048576u
int im_gae_static(const float *rew, const float *cost, const float *val, const uint8_t *done, float *adv, float *ret,
                  double *sum_cost, uint32_t n_ticks, uint32_t n_envs, float gamma, float lambda, float lagrange_mu,
                  void *cuda_stream, char *errbuf, size_t errbuf_bytes);

void im_destroy(im_ctx *ctx);

/* Message of the last failing call on this ctx (string owned by ctx, valid until the next call); "" if none.
 * With ctx == NULL: message of the last failing im_create / im_arena_bytes on this thread. */
const char *im_last_error(const im_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* INFRAMIND_H */
