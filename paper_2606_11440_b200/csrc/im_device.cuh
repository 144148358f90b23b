// im_device.cuh — device-side parameter block, HBM state layout and the small defined functions (Philox, im_exp,
// im_tanh) of the CUDA path.  Written independently of oracle/ (no shared code); the definitions follow
// DESIGN.md readings R2, R3, R23, R24.
//
// HBM layout of the environment state.  Environments are grouped in BLOCKS of 32: block b
// holds envs 32b .. 32b+31 and is owned by ONE WARP of the simulation kernel, lane = env & 31 (one thread per env).
// A block is one contiguous record (stride multiple of 128 B):
//   [ hdr | cm | kvt | ctr | hot | iss | qready |  cold[32] | wkey[32] | waux[32] | q[32] ]
// The first seven parts are struct-of-arrays ACROSS the 32 envs of the block ("SoA-32"): unit u of lane l sits at
// part + (u * 32 + l) * unit_bytes, so that a warp whose lanes walk their own envs in step reads and writes whole
// 128 .. 512-byte lines, and the header lands in shared memory as [word][lane] (bank = lane: conflict-free for any
// word index) with ONE bulk copy (cp.async.bulk) per block.  The last four parts are per-env arrays (lane l at
// part + l * stride): they are touched only at data-dependent positions by the few requests that change state.
//   hdr   u32 units (hdr_words): m[3k] = n_wait | n_run << 16, m[3k+1] = kv_used, m[3k+2] = ewma_q8 |
//         occ (bit gs = global slot gs taken; SP bits + two padding words) | qfree[QW] | the chunk directory of the waiting
//         lists: next[c] (one byte per chunk, 0xFF = end: every model's chunks and the free chunks are linked lists) |
//         head[k] (one byte per model, 0xFF = empty) | misc0 = drops | free head << 16 |
//         misc1 = icnt
//   cm    u32 units (cm_words): completion bytes of the tick's service pass, one per slot group (k_serve -> k_sim)
//   kvt   u32 units (N): tokens decoded per model by the tick's service pass (k_serve -> k_sim)
//   ctr   u32 units (16): the counters of enum Counter (absolute ticks < 65536 keep every sum below 2^32)
//   hot   uint4 units (SP / 8): remaining tokens of the 8 slots of a group as 8 x u16 (slot 2j = low half of word j);
//         a FREE slot holds 0, so the service pass needs no occupancy bits.  SP = sum_k ceil8(S_k): the slots of all
//         models numbered consecutively (R10); a group belongs to ONE model and to ONE Philox call (R2)
//   iss   uint2 units (kIssueCap): {key, static word} written by the executor kernel for this tick (phase D)
//   qready u32 units (QW): queries whose next stage is due, kept only ACROSS im_rollout calls
//   cold[gs] 32 bytes = {issue(16) | deadline<<16, sw, id, 0, 0, 0, 0, 0}: written whole (st256) at admission
//         sw = out_total(13) | in_tok(13)<<13 | succ<<26 | depth<<27
//   wkey[c][32], waux[c][32]: the waiting lists, ONE UNORDERED LIST PER MODEL built from chunks of 32 entries out of a
//         pool of n_chunks = RCAP/32 + N per env (only the head chunk of a model is partly filled, so the pool
//         always suffices): admission only reads the chunks of the model that admits.  key = model<<28 |
//         time(16)<<12 | id, time = deadline (EDF) or issue tick (FCFS): one u32 compare is the R20 order; id =
//         4*query + agent.  A list of n entries fills its non-head chunks and the first ((n - 1) & 31) + 1 entries of
//         its head chunk; the rest of the head chunk holds 0xFFFFFFFF (never a valid key): a chunk is written whole
//         when it is taken from the pool.
//         waux = {issue(16) | remaining<<16, sw}
//   q[i]     uint4 = {plan word, budget | in_tok<<16, deadline, arrive}
// Free query slots are defined by the qfree bitmap and free service slots by occ (their cold words hold stale data).
// Absolute ticks are < 65536 on the device.
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>

namespace im {

constexpr uint32_t kMaxModels = 16;
constexpr uint32_t kRegions = 64;        // row-list / log regions (one atomic counter each), region = (env / 32) % n_regions
constexpr uint32_t kDtUs = 50000;
constexpr uint32_t kCntStride = 32;      // words between the append counters of two regions: one 128-byte line each, so that
                                         // the claims of different regions never queue on the same L2 line
constexpr uint32_t kChunk = 32;          // entries per waiting-list chunk
constexpr uint32_t kIssueCap = 128;      // issue records per env per tick (31 arrivals x 3 calls + continuing stages)

constexpr uint32_t ST_FREE = 0, ST_WAIT = 1, ST_RUN = 2;
constexpr uint32_t SW_IN_SHIFT = 13, SW_SUCC_SHIFT = 26, SW_DEPTH_SHIFT = 27, SW_TOK_MASK = 0x1FFFu;
// query plan word: live0 planned1 topo2-3 cnt4-5 keff6-8 stage9-11 nst12-14 pending15-16 solved17 roles18-25
constexpr uint32_t QP_LIVE = 1u, QP_PLANNED = 2u;
constexpr uint32_t QP_PEND_SHIFT = 15, QP_SUCC_SHIFT = 17, QP_ROLE_SHIFT = 18;

enum Stream : uint32_t { STREAM_ARR = 1, STREAM_QRY = 2, STREAM_PLAN = 3, STREAM_EXEC = 4, STREAM_SVC = 5 };
enum Counter : uint32_t { C_ARRIVALS, C_DROPPED, C_FINISHED, C_SOLVED, C_MISSED, C_ISSUED, C_CALLS_DONE, C_PREEMPT,
                          C_SUM_SOJOURN, C_SUM_LIVE_MID, C_PLANS, C_EXEC_DEC, C_SUM_RUNNING, C_SUM_WAITING, C_NEAR,
                          C_ABANDONED, C_N };

struct ModelTab {
    uint32_t rate, slots, kv_cap, prefill;
    uint32_t succ[3];
    float kv_inv;
};

// a work list that doubles as the decision log: 64 regions, each a ring of `regcap` rows
//   row = { env (local), a, deadline, in_tok | result<<16 }
//   a (exec) = q | agent<<10 | topo<<12 | role<<14 | keff<<16 | t_rel<<19 ; a (plan) = q | t_rel<<19
//   result (exec) = action ; result (plan) = topo | cnt<<2 | roles<<4
struct RowBuf {
    uint4 *row;
    float *logp;
    float *val;          // exec only
    float *logits;       // optional [rows][n_out]
    uint32_t *cnt;       // [kRegions * kCntStride] monotonically increasing append counters, counter of region r at r * kCntStride
    uint32_t *base;      // [2][kRegions] start of the current tick's rows (parity double buffer)
    uint32_t regcap;
    uint32_t n_out;
};

struct QLog {
    uint4 *rec;          // {env (global), arrive, sojourn, budget | solved<<16 | topo<<17 | keff<<19}
    float *unorm;
    uint32_t *cnt;       // [kRegions * kCntStride], as RowBuf::cnt
    uint32_t regcap;
};

struct Params {
    uint32_t E, N, QCAP, RCAP, QW, SP;                 // SP = padded slot count of the pool
    uint32_t NB, n_regions;                            // 32-env blocks; row-list regions in use = min(kRegions, NB)
    uint32_t sched_mode, kv_preempt, cost_mode, episode_ticks, budget_norm, in_tok_const, mix_thresh, env_id_base;
    uint32_t mix_lo[2], mix_hi[2], depth_median[3];
    uint32_t flags, has_intok, seed_lo, seed_hi;
    uint32_t f_in, hidden, log_mode, pad0;
    ModelTab model[kMaxModels];
    uint32_t slot_base[kMaxModels + 1];      // first global slot of each model (multiples of 8)
    uint32_t svc_rk[20];                     // Philox round keys of the service stream (k0, k1 per round): constant-bank operands
    // env state: one record per block of 32 envs (layout at the top of this file)
    uint8_t *env_base;
    unsigned long long blk_stride;           // bytes, multiple of 128
    uint32_t hw_occ, hw_qfree, hw_next, hw_head, hw_misc, hdr_words;   // header word indices (m at word 0)
    uint32_t off_cm, off_kvt, off_ctr, off_hot, off_iss, off_qready;      // SoA-32 parts: byte offsets inside the block (hdr at 0)
    uint32_t off_cold, off_wkey, off_waux, off_q, cold_stride, wkey_stride, waux_stride, q_stride;   // per-env parts: lane 0 and lane stride
    uint32_t n_grp, cm_words;                // SP / 8 slot groups; completion-mask words per env = ceil(n_grp / 4)
    uint32_t n_chunks;                       // waiting-list chunks per env: RCAP / 32 + N (< 255: chunk ids are bytes)
    float *snap;                             // [E][3N] telemetry features of the current tick (R14)
    const uint32_t *tab_mult, *tab_intok, *tab_cdf;
    const uint8_t *env_level;
    float *rew, *cost, *val;
    uint8_t *done, *miss;
    RowBuf exec, plan;
    QLog qlog;
    uint32_t *err_flag;
};

struct Weights {          // device copies of one net, prepared by k_repack (im_api.cu)
    const float *W1t, *W2t, *W3t;        // fp32 path: transposed [k][o]; W3t has ld = n_out_pad
    const __nv_bfloat16 *W1, *W2, *W3;   // bf16 path: [o][k] row-major, W3 zero-padded to n_out_pad rows
    const float *b1, *b2, *b3;           // fp32 biases (b3 padded)
    uint32_t n_out, n_out_pad;
    uint8_t *tc_img;                     // bf16 nets (tcgen05 path): shared-memory image of the net (im_tc.cuh), else null
};

__device__ __forceinline__ uint8_t *blk_rec(const Params &P, uint32_t e) { return P.env_base + (size_t)(e >> 5) * P.blk_stride; }
// word w of env e's header (SoA-32: [word][lane])
__device__ __forceinline__ uint32_t *hdr_word(const Params &P, uint32_t e, uint32_t w)
{
    return reinterpret_cast<uint32_t *>(blk_rec(P, e)) + w * 32u + (e & 31u);
}
__device__ __forceinline__ uint2 *iss_rec(const Params &P, uint32_t e, uint32_t slot)
{
    return reinterpret_cast<uint2 *>(blk_rec(P, e) + P.off_iss) + slot * 32u + (e & 31u);
}
__device__ __forceinline__ uint4 *env_q(const Params &P, uint32_t e)
{
    return reinterpret_cast<uint4 *>(blk_rec(P, e) + P.off_q + (size_t)(e & 31u) * P.q_stride);
}
// A 32-byte record written with ONE 256-bit store is a full-sector write: the memory system takes it as one DRAM
// transaction, where a narrower store to a sector that is not resident costs a fill read plus the write (measured:
// 44 G/s against 22.6 G/s for random sectors).  The per-request records that are written at
// data-dependent positions (running-slot records) are therefore 32 bytes and 32-byte aligned.
__device__ __forceinline__ void st256(void *p, uint4 a, uint4 b)
{
    asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(p), "r"(a.x), "r"(a.y), "r"(a.z), "r"(a.w), "r"(b.x),
                 "r"(b.y), "r"(b.z), "r"(b.w)
                 : "memory");
}
// row-list / log region of an env: the 32 envs of a block share one, so that a warp claims rows with one atomic
__device__ __forceinline__ uint32_t region_of(const Params &P, uint32_t e) { return (e >> 5) % P.n_regions; }

// ------------------------------------------------------------------------------------------------ R2
struct Ph4 { uint32_t x, y, z, w; };

__device__ __forceinline__ Ph4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; r++) {
        const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0, p1 = (unsigned long long)0xCD9E8D57u * c2;   // IMAD.WIDE
        c0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0; c1 = (uint32_t)p1;
        c2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1; c3 = (uint32_t)p0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return Ph4{c0, c1, c2, c3};
}

// the same with the 10 round keys precomputed (k_r = k + r * Weyl): saves the two key additions of every round
__device__ __forceinline__ Ph4 philox4x32_10_rk(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const uint32_t (&rk)[20])
{
#pragma unroll
    for (int r = 0; r < 10; r++) {
        const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0, p1 = (unsigned long long)0xCD9E8D57u * c2;
        c0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk[2 * r]; c1 = (uint32_t)p1;
        c2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk[2 * r + 1]; c3 = (uint32_t)p0;
    }
    return Ph4{c0, c1, c2, c3};
}

__device__ __forceinline__ Ph4 draw(const Params &P, uint32_t stream, uint32_t gid, int32_t t, uint32_t slot, uint32_t sub)
{
    return philox4x32_10(gid, (uint32_t)t, slot, sub, P.seed_lo, P.seed_hi ^ stream);
}

// R3: u = (x >> 8) * 2^-24
__device__ __forceinline__ float u24(uint32_t x) { return __uint2float_rn(x >> 8) * 0x1p-24f; }

// ----------------------------------------------------------------------------------------------- R23
__device__ __forceinline__ float im_exp(float x)
{
    // branch-free (the x < -80 case is a select at the end): 48 of these per executor decision must interleave, and an
    // early return keeps the compiler from overlapping their dependent chains (measured: 8600 -> cycles per tile)
    // n = rintf(x log2e) without the conversion unit: adding 1.5 * 2^23 rounds to an integer (RNE, |x log2e| < 2^22) and
    // leaves that integer in the low bits of the sum; 2^n is then an add into the exponent field of p (exact: the
    // result is normal for n >= -116).  Same values as rintf / ldexpf, two FADDs and two integer ops.
    const float t = __fadd_rn(__fmul_rn(x, 0x1.715476p+0f), 12582912.0f);
    const float n = __fsub_rn(t, 12582912.0f);
    float r = __fmaf_rn(n, -0x1.62e400p-1f, x);
    r = __fmaf_rn(n, -0x1.7f7d1cp-20f, r);
    float p = 0x1.6c16c2p-10f;
    p = __fmaf_rn(p, r, 0x1.111112p-7f);
    p = __fmaf_rn(p, r, 0x1.555556p-5f);
    p = __fmaf_rn(p, r, 0x1.555556p-3f);
    p = __fmaf_rn(p, r, 0.5f);
    p = __fmaf_rn(p, r, 1.0f);
    p = __fmaf_rn(p, r, 1.0f);
    const float y = __int_as_float(__float_as_int(p) + (__float_as_int(t) << 23));   // p * 2^n (the low 9 bits of the magic are 0)
    return x < -80.0f ? 0.0f : y;
}

// Two im_exp at once with the packed fp32 instructions of sm_100 (mul / add / fma .f32x2: each half rounds exactly like
// the scalar operation, so the values are those of im_exp bit for bit); 19 instructions per pair instead of 32.
struct F2 { unsigned long long v; };
__device__ __forceinline__ F2 f2_pack(float a, float b) { F2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void f2_unpack(F2 p, float &a, float &b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(p.v)); }
__device__ __forceinline__ F2 f2_mul(F2 a, F2 b) { F2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ F2 f2_add(F2 a, F2 b) { F2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ F2 f2_fma(F2 a, F2 b, F2 c) { F2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v)); return r; }
__device__ __forceinline__ void im_exp_x2(float x0, float x1, float &y0, float &y1)
{
    const F2 x = f2_pack(x0, x1), magic = f2_pack(12582912.0f, 12582912.0f), nmagic = f2_pack(-12582912.0f, -12582912.0f);
    const F2 t = f2_add(f2_mul(x, f2_pack(0x1.715476p+0f, 0x1.715476p+0f)), magic);
    const F2 n = f2_add(t, nmagic);                                   // t - magic == t + (-magic), exactly
    F2 r = f2_fma(n, f2_pack(-0x1.62e400p-1f, -0x1.62e400p-1f), x);
    r = f2_fma(n, f2_pack(-0x1.7f7d1cp-20f, -0x1.7f7d1cp-20f), r);
    F2 p = f2_pack(0x1.6c16c2p-10f, 0x1.6c16c2p-10f);
    p = f2_fma(p, r, f2_pack(0x1.111112p-7f, 0x1.111112p-7f));
    p = f2_fma(p, r, f2_pack(0x1.555556p-5f, 0x1.555556p-5f));
    p = f2_fma(p, r, f2_pack(0x1.555556p-3f, 0x1.555556p-3f));
    p = f2_fma(p, r, f2_pack(0.5f, 0.5f));
    p = f2_fma(p, r, f2_pack(1.0f, 1.0f));
    p = f2_fma(p, r, f2_pack(1.0f, 1.0f));
    float p0, p1, t0, t1;
    f2_unpack(p, p0, p1); f2_unpack(t, t0, t1);
    const float z0 = __int_as_float(__float_as_int(p0) + (__float_as_int(t0) << 23));
    const float z1 = __int_as_float(__float_as_int(p1) + (__float_as_int(t1) << 23));
    y0 = x0 < -80.0f ? 0.0f : z0;
    y1 = x1 < -80.0f ? 0.0f : z1;
}

__device__ __forceinline__ float im_tanh(float x)
{
    const float e = im_exp(__fmul_rn(-2.0f, fabsf(x)));
    const float q = __fdiv_rn(__fsub_rn(1.0f, e), __fadd_rn(1.0f, e));
    return copysignf(q, x);
}

// ----------------------------------------------------------------------------------------------- R17
__device__ __forceinline__ uint32_t keff_of(uint32_t topo, uint32_t K) { return topo == 0 ? 1u : (topo == 1 ? K : (K < 2 ? 2u : K)); }
__device__ __forceinline__ uint32_t nstages_of(uint32_t topo, uint32_t keff) { return topo == 0 ? 1u : (topo == 1 ? keff : 2u); }
__device__ __forceinline__ void stage_calls(uint32_t topo, uint32_t keff, uint32_t stage, uint32_t &a0, uint32_t &nc)
{
    if (topo == 0) { a0 = 0; nc = 1; }
    else if (topo == 1) { a0 = stage; nc = 1; }
    else if (topo == 2) { if (stage == 0) { a0 = 0; nc = keff - 1; } else { a0 = keff - 1; nc = 1; } }
    else { if (stage == 0) { a0 = 0; nc = 1; } else { a0 = 1; nc = keff - 1; } }
}

__device__ __forceinline__ uint32_t row_gid(const RowBuf &rb, uint32_t region, uint32_t idx) { return region * rb.regcap + (idx % rb.regcap); }
// the same for base + j with base already reduced modulo regcap and j <= regcap (one division per claim, not per row)
__device__ __forceinline__ uint32_t row_gid_wrapped(const RowBuf &rb, uint32_t region, uint32_t base_mod, uint32_t j)
{
    uint32_t r = base_mod + j;
    if (r >= rb.regcap) r -= rb.regcap;
    return region * rb.regcap + r;
}

// claim n consecutive rows of region `region`.  In log mode the region is a linear log of the rollout and an overflow is
// flagged here; without the log it is a ring that only has to hold one tick's rows, and the consumer (sched_init of
// im_policy.cu) flags a tick that produced more rows than the ring holds.
__device__ __forceinline__ uint32_t rows_claim(const Params &P, const RowBuf &rb, uint32_t region, uint32_t n)
{
    const uint32_t idx = atomicAdd(&rb.cnt[region * kCntStride], n);
    if (P.log_mode && idx + n > rb.regcap) atomicOr(P.err_flag, 1u);
    return idx;
}

// executor rows of one stage of query q (R17); `pw` is the query's plan word with stage = the stage to dispatch;
// idx0 is the claimed ring position already reduced modulo regcap
__device__ __forceinline__ void write_exec_rows(const Params &P, uint32_t region, uint32_t idx0, uint32_t e, uint32_t q, uint32_t pw,
                                                uint32_t in_tok, int32_t dl, uint32_t t_rel, uint32_t a0, uint32_t nc)
{
    const uint32_t topo = (pw >> 2) & 3u, keff = (pw >> 6) & 7u, roles = (pw >> QP_ROLE_SHIFT) & 0xFFu;
#pragma unroll 1
    for (uint32_t j = 0; j < nc; j++) {
        const uint32_t agent = a0 + j;
        const uint32_t a = q | (agent << 10) | (topo << 12) | (((roles >> (2 * agent)) & 3u) << 14) | (keff << 16) | (t_rel << 19);
        P.exec.row[row_gid_wrapped(P.exec, region, idx0, j)] = make_uint4(e, a, (uint32_t)dl, in_tok);
    }
}

// ------------------------------------------------------------------------------------ chained launches
// The kernels of a tick (planner, executor, k_serve, k_sim) depend on each other in stream order.  They are launched
// with programmatic stream serialisation: the successor's CTAs are set up while the predecessor drains and run their own
// prologue - weight image into shared memory, tensor-memory allocation, tables - before they wait (griddep_wait) until
// the predecessor grid has completed and its writes are visible: +1.3 % on the whole step.  No kernel triggers its
// successor early (griddepcontrol.launch_dependents at the top of the policy kernels / k_sim / all of them: -1.2 % /
// -0.3 % / -8 %: the early CTAs take the places of the predecessor's own).  Rules: every CTA executes griddep_wait
// before it returns (so "my predecessor is complete" is transitive along the chain), and nothing before the wait reads
// what a kernel of the same rollout writes.
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <typename... KArgs, typename... Args>
static inline cudaError_t launch_chained(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool chained, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = chained ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ------------------------------------------------------------------------------------ bulk async copies (TMA, 1-D)
// One elected lane moves a whole header block between HBM and shared memory; completion of a load is signalled on an
// mbarrier (complete_tx), completion of a store through the bulk async-group.  Sizes and addresses are multiples of 16 B.
namespace bulk {
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n\t"
        ".reg .pred P1;\n\t"
        "BULK_WAIT:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
        "@P1 bra BULK_DONE;\n\t"
        "bra BULK_WAIT;\n\t"
        "BULK_DONE:\n\t"
        "}" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
__device__ __forceinline__ void g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void s2g(void *dst_gmem, const void *src_smem, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
// the source (shared memory) of every committed bulk store has been read: enough before the CTA exits, the end of the
// kernel orders the writes themselves
__device__ __forceinline__ void wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
}  // namespace bulk

}  // namespace im
