// im_policy.cu — batched planner / executor / critic MLP forward + inverse-CDF sampling (R15-R26).
//
// Work comes as row lists written by k_sim (and, for stage 0 of new queries, by the planner kernel itself);
// the executor launch also evaluates one critic row per env (R30).  Two numerics contracts:
//   fp32 (R22): y = b; for k ascending: y = fmaf(W[o][k], x[k], y); tanh = im_tanh  -> bit-exact vs the oracle.
//   bf16 (R25): bf16 operands, fp32 accumulation on the tensor cores (tcgen05, accumulators in tensor memory),
//               tanh.approx, fp32 logits; sampling by the exact R24 sampler on those logits.
#include "im_device.cuh"
#include "im_tc.cuh"
#include <cuda_bf16.h>

namespace im {

struct RowInfo { uint32_t env, a, c; int32_t dl; float b; uint32_t gidx; bool critic; };

// ------------------------------------------------------------------------------------------------ tiles
struct TileSched {
    uint32_t pref[kRegions + 1];
    uint32_t base[kRegions];
    uint32_t cnt[kRegions];      // append counters at kernel start (the kernel's own list does not grow while it runs)
    uint32_t base_mod[kRegions]; // base % regcap: the ring position of the region's first row of this tick
    uint32_t crit_tiles, total;
};

__device__ __forceinline__ void sched_init(const Params &P, TileSched &S, const RowBuf &rb, uint32_t parity, uint32_t rows_per_tile, uint32_t n_crit)
{
    if (threadIdx.x < kRegions) {
        const uint32_t b = rb.base[parity * kRegions + threadIdx.x], c = rb.cnt[threadIdx.x * kCntStride];
        // a ring (no decision log) holds one tick's rows: more than regcap of them have overwritten each other
        if (blockIdx.x == 0 && !P.log_mode && c - b > rb.regcap) atomicOr(P.err_flag, 1u);
        S.base[threadIdx.x] = b;
        S.cnt[threadIdx.x] = c;
        S.base_mod[threadIdx.x] = b % rb.regcap;
        S.pref[threadIdx.x + 1] = (c - b + rows_per_tile - 1) / rows_per_tile;
        if (blockIdx.x == 0) rb.base[(parity ^ 1u) * kRegions + threadIdx.x] = c;   // next tick starts here
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        S.crit_tiles = (n_crit + rows_per_tile - 1) / rows_per_tile;
        S.pref[0] = 0;
        for (uint32_t r = 0; r < kRegions; r++) S.pref[r + 1] += S.pref[r];
        S.total = S.crit_tiles + S.pref[kRegions];
    }
    __syncthreads();
}

// row `r` of tile `tile`: fills info, returns false if out of range
template <bool EXEC>
__device__ __forceinline__ bool tile_row(const Params &P, const TileSched &S, const RowBuf &rb, uint32_t tile, uint32_t r, uint32_t rows_per_tile,
                                         uint32_t n_crit, int32_t t0, RowInfo &ri)
{
    if (tile < S.crit_tiles) {
        const uint32_t env = tile * rows_per_tile + r;
        if (env >= n_crit) return false;
        ri.env = env; ri.a = 0; ri.c = 0; ri.dl = 0; ri.b = 0.0f; ri.gidx = 0; ri.critic = true;
        return true;
    }
    const uint32_t lt = tile - S.crit_tiles;
    uint32_t lo = 0, hi = kRegions;
    while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if (S.pref[mid] <= lt) lo = mid; else hi = mid; }
    const uint32_t idx = S.base[lo] + (lt - S.pref[lo]) * rows_per_tile + r;
    if (idx >= S.cnt[lo]) return false;
    const uint32_t g = row_gid(rb, lo, idx);
    const uint4 row = rb.row[g];
    ri.env = row.x; ri.a = row.y; ri.dl = (int32_t)row.z; ri.c = row.w; ri.gidx = g; ri.critic = false;
    // budget feature (R15): planner b = budget / norm (the row is created at the arrival tick, deadline - t = budget);
    // executor b = clamp((deadline - t) / norm, -1, 1) ("normalized remaining budget")
    const int32_t t = t0 + (int32_t)(row.y >> 19);
    float b = __fdiv_rn(__int2float_rn(ri.dl - t), __uint2float_rn(P.budget_norm));
    if (EXEC) b = fminf(fmaxf(b, -1.0f), 1.0f);
    ri.b = b;
    return true;
}

// feature k of a row (R15)
__device__ __forceinline__ float feature(const Params &P, bool exec, const RowInfo &ri, uint32_t k)
{
    const uint32_t N3 = 3 * P.N;
    if (k == 0) return ri.b;
    if (k <= N3) return P.snap[(size_t)ri.env * N3 + (k - 1)];
    if (ri.critic) return 0.0f;
    if (k == N3 + 1) return __uint2float_rn(ri.c & 0xFFFFu) * 0x1p-13f;
    if (!exec) return 0.0f;
    const uint32_t j = k - (N3 + 2);
    if (j < 4) return j == ((ri.a >> 12) & 3u) ? 1.0f : 0.0f;
    if (j < 8) return (j - 4) == ((ri.a >> 14) & 3u) ? 1.0f : 0.0f;
    if (j == 8) return __uint2float_rn((ri.a >> 10) & 3u) * 0.25f;
    if (j == 9) return __uint2float_rn((ri.a >> 16) & 7u) * 0.25f;
    return 0.0f;
}

// ------------------------------------------------------------------------------------------- epilogues
// sequential R24 sampler over logits l[0..n) (shared memory); e[] is scratch of n floats
__device__ __forceinline__ uint32_t sample_seq(const float *l, float *e, uint32_t n, float u, float &logp)
{
    float m = l[0];
    for (uint32_t i = 1; i < n; i++) m = fmaxf(m, l[i]);
    float Z = 0.0f;
    for (uint32_t i = 0; i < n; i++) { const float v = im_exp(__fsub_rn(l[i], m)); e[i] = v; Z = __fadd_rn(Z, v); }
    const float th = __fmul_rn(u, Z);
    uint32_t a = n - 1;
    float c = 0.0f;
    for (uint32_t i = 0; i < n; i++) { c = __fadd_rn(c, e[i]); if (c > th) { a = i; break; } }
    logp = __fsub_rn(__fsub_rn(l[a], m), logf(Z));
    return a;
}

// executor decision -> log row + one issue record of its env (R18): {waiting-list key, static word} (im_device.cuh);
// phase D of the simulation kernel appends it to the env's waiting list.
// `slot_in` != ~0u: issue-list slot of the env already claimed by the caller (claimed early to hide the atomic's latency)
__device__ __forceinline__ void exec_commit(const Params &P, const RowInfo &ri, const Ph4 &d, uint32_t act, float logp, float value, int32_t t,
                                            uint32_t slot_in = ~0u)
{
    const uint32_t q = ri.a & 0x3FFu, agent = (ri.a >> 10) & 3u;
    if (P.log_mode) {
        P.exec.row[ri.gidx].w = (ri.c & 0xFFFFu) | (act << 16);
        P.exec.logp[ri.gidx] = logp;
        P.exec.val[ri.gidx] = value;
    }
    const uint32_t model = act / 3u, depth = act - model * 3u;
    uint32_t out_total = (uint32_t)(((unsigned long long)P.depth_median[depth] * __ldg(&P.tab_mult[d.y >> 22])) >> 16);
    out_total = out_total < 1u ? 1u : out_total;
    const uint32_t succ = d.z < P.model[model].succ[depth] ? 1u : 0u;
    const uint32_t slot = slot_in != ~0u ? slot_in : atomicAdd(hdr_word(P, ri.env, P.hw_misc + 1u), 1u);
    const uint32_t tm = (uint32_t)(P.sched_mode ? ri.dl : t) & 0xFFFFu;             // R20: deadline (EDF) or issue tick (FCFS)
    if (slot < kIssueCap)
        *iss_rec(P, ri.env, slot) =
            make_uint2((model << 28) | (tm << 12) | (q << 2) | agent,
                       out_total | ((ri.c & 0xFFFFu) << SW_IN_SHIFT) | (succ << SW_SUCC_SHIFT) | (depth << SW_DEPTH_SHIFT));
    else
        atomicOr(P.err_flag, 4u);
}

// executor / critic row: logits[0..3N) + value at 3N (shared-memory logits, sequential R24 sampler)
__device__ __forceinline__ void exec_epilogue(const Params &P, const RowInfo &ri, const float *logits, float *scratch,
                                              int32_t t0, uint32_t trow)
{
    const uint32_t n = 3 * P.N;
    const float value = logits[n];
    if (ri.critic) { P.val[(size_t)trow * P.E + ri.env] = value; return; }
    const uint32_t q = ri.a & 0x3FFu, agent = (ri.a >> 10) & 3u;
    const int32_t t = t0 + (int32_t)(ri.a >> 19);
    if (P.exec.logits) for (uint32_t i = 0; i <= n; i++) P.exec.logits[(size_t)ri.gidx * P.exec.n_out + i] = logits[i];
    const Ph4 d = draw(P, STREAM_EXEC, P.env_id_base + ri.env, t, q * 4u + agent, 0);
    float logp;
    const uint32_t act = sample_seq(logits, scratch, n, u24(d.x), logp);
    exec_commit(P, ri, d, act, logp, value, t);
}

// planner decision -> log row, plan word of the query and the stage-0 executor rows (R17)
// claimed_idx0 != ~0u: ring position (reduced modulo regcap) of the row's stage-0 executor rows, claimed by the caller
__device__ __forceinline__ void plan_commit(const Params &P, const RowInfo &ri, uint32_t topo, uint32_t cnt, uint32_t roles, float lp,
                                            uint32_t claimed_idx0 = ~0u)
{
    const uint32_t q = ri.a & 0x3FFu, t_rel = ri.a >> 19;
    const uint32_t keff = keff_of(topo, cnt + 1), nst = nstages_of(topo, keff);
    if (P.log_mode) {
        P.plan.row[ri.gidx].w = (ri.c & 0xFFFFu) | ((topo | (cnt << 2) | (roles << 4)) << 16);
        P.plan.logp[ri.gidx] = lp;
    }
    // stage 0 executor rows; the plan word records stage = 1, pending = calls of stage 0 (issued in phase D of this tick)
    uint32_t a0, nc;
    stage_calls(topo, keff, 0, a0, nc);
    const uint32_t pw = QP_LIVE | QP_PLANNED | (topo << 2) | (cnt << 4) | (keff << 6) | (nst << 12) | (roles << QP_ROLE_SHIFT);
    env_q(P, ri.env)[q].x = pw | (1u << 9) | (nc << QP_PEND_SHIFT);
    const uint32_t region = region_of(P, ri.env);
    const uint32_t idx0 = claimed_idx0 != ~0u ? claimed_idx0 : rows_claim(P, P.exec, region, nc) % P.exec.regcap;
    write_exec_rows(P, region, idx0, ri.env, q, pw, ri.c & 0xFFFFu, ri.dl, t_rel, a0, nc);
}

// planner row: 24 logits = [4 topology | 4 count | 4 agents x 4 roles] (R16)
__device__ __forceinline__ void plan_epilogue(const Params &P, const RowInfo &ri, const float *logits, float *scratch, int32_t t0)
{
    const uint32_t q = ri.a & 0x3FFu, t_rel = ri.a >> 19;
    const int32_t t = t0 + (int32_t)t_rel;
    const uint32_t gid = P.env_id_base + ri.env;
    if (P.plan.logits) for (uint32_t i = 0; i < 24; i++) P.plan.logits[(size_t)ri.gidx * 24 + i] = logits[i];
    const Ph4 d0 = draw(P, STREAM_PLAN, gid, t, q, 0), d1 = draw(P, STREAM_PLAN, gid, t, q, 1);
    float lp_t, lp_c, lp_r[4];
    const uint32_t topo = sample_seq(logits, scratch, 4, u24(d0.x), lp_t);
    const uint32_t cnt = sample_seq(logits + 4, scratch, 4, u24(d0.y), lp_c);
    const uint32_t ur[4] = {d1.x, d1.y, d1.z, d1.w};
    uint32_t roles = 0;
#pragma unroll
    for (uint32_t a = 0; a < 4; a++) roles |= sample_seq(logits + 8 + 4 * a, scratch, 4, u24(ur[a]), lp_r[a]) << (2 * a);
    const uint32_t keff = keff_of(topo, cnt + 1);
    float lp = __fadd_rn(lp_t, lp_c);
#pragma unroll
    for (uint32_t a = 0; a < 4; a++) if (a < keff) lp = __fadd_rn(lp, lp_r[a]);
    plan_commit(P, ri, topo, cnt, roles, lp);
}

// ================================================================================================ fp32 path (R22)
constexpr int kF32Warps = 8, kF32RowsPerWarp = 4, kF32Rows = kF32Warps * kF32RowsPerWarp;

template <bool EXEC>
__global__ void __launch_bounds__(kF32Warps * 32)
k_policy_f32(const Params P, const Weights W, uint32_t parity, int32_t t0, uint32_t trow)
{
    extern __shared__ __align__(16) float smem_f[];
    __shared__ TileSched sched;
    const uint32_t F = P.f_in, H = P.hidden, NO = W.n_out, NOP = W.n_out_pad;
    float *sW1 = smem_f, *sW2 = sW1 + F * H, *sW3 = sW2 + H * H, *sb1 = sW3 + H * NOP, *sb2 = sb1 + H, *sb3 = sb2 + H;
    float *sx = sb3 + NOP;                               // per warp: [4][F] + [4][H] + [4][H] + [4][64] logits + [4][64] scratch
    // The weights come by bulk async copies (TMA 1-D) that one thread issues and that fly while the CTA builds its tile
    // schedule.  (Copied by a loop of scalar loads and stores they were 80 % of the kernel's time on the small
    // configurations: ptxas does not overlap the loads of such a loop, 32 dependent L2 round trips per launch.)
    __shared__ uint64_t wbar;
    if (threadIdx.x == 0) {
        bulk::mbar_init(&wbar, 1);
        bulk::fence_mbar_init();
        bulk::mbar_expect_tx(&wbar, 4u * (F * H + H * H + H * NOP + 2u * H + NOP));
        auto copy = [&](float *dst, const float *src, uint32_t n_floats) {       // sizes and addresses are multiples of 16 bytes
            constexpr uint32_t kPiece = 32 * 1024;
            for (uint32_t o = 0; o < 4u * n_floats; o += kPiece)
                bulk::g2s(reinterpret_cast<uint8_t *>(dst) + o, reinterpret_cast<const uint8_t *>(src) + o, min(kPiece, 4u * n_floats - o), &wbar);
        };
        copy(sW1, W.W1t, F * H); copy(sW2, W.W2t, H * H); copy(sW3, W.W3t, H * NOP);
        copy(sb1, W.b1, H); copy(sb2, W.b2, H); copy(sb3, W.b3, NOP);
    }
    const RowBuf &rb = EXEC ? P.exec : P.plan;
    const uint32_t n_crit = EXEC ? P.E : 0u;
    sched_init(P, sched, rb, parity, kF32Rows, n_crit);
    bulk::mbar_wait(&wbar, 0);

    const uint32_t lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const uint32_t per_warp = kF32RowsPerWarp * (F + 2 * H + 128);
    float *x = sx + wib * per_warp, *h1 = x + kF32RowsPerWarp * F, *h2 = h1 + kF32RowsPerWarp * H, *lg = h2 + kF32RowsPerWarp * H;
    float *scr = lg + kF32RowsPerWarp * 64;

    for (uint32_t tile = blockIdx.x; tile < sched.total; tile += gridDim.x) {
        RowInfo ri[kF32RowsPerWarp];
        bool ok[kF32RowsPerWarp];
#pragma unroll
        for (int r = 0; r < kF32RowsPerWarp; r++) {
            ok[r] = tile_row<EXEC>(P, sched, rb, tile, wib * kF32RowsPerWarp + r, kF32Rows, n_crit, t0, ri[r]);
            for (uint32_t k = lane; k < F; k += 32) x[r * F + k] = ok[r] ? feature(P, EXEC, ri[r], k) : 0.0f;
        }
        __syncwarp();
        if (!(ok[0] | ok[1] | ok[2] | ok[3])) continue;
        for (uint32_t o = lane; o < H; o += 32) {
            float acc[kF32RowsPerWarp];
#pragma unroll
            for (int r = 0; r < kF32RowsPerWarp; r++) acc[r] = sb1[o];
            for (uint32_t k = 0; k < F; k++) {
                const float w = sW1[k * H + o];
#pragma unroll
                for (int r = 0; r < kF32RowsPerWarp; r++) acc[r] = __fmaf_rn(w, x[r * F + k], acc[r]);
            }
#pragma unroll
            for (int r = 0; r < kF32RowsPerWarp; r++) h1[r * H + o] = im_tanh(acc[r]);
        }
        __syncwarp();
        for (uint32_t o = lane; o < H; o += 32) {
            float acc[kF32RowsPerWarp];
#pragma unroll
            for (int r = 0; r < kF32RowsPerWarp; r++) acc[r] = sb2[o];
            for (uint32_t k = 0; k < H; k++) {
                const float w = sW2[k * H + o];
#pragma unroll
                for (int r = 0; r < kF32RowsPerWarp; r++) acc[r] = __fmaf_rn(w, h1[r * H + k], acc[r]);
            }
#pragma unroll
            for (int r = 0; r < kF32RowsPerWarp; r++) h2[r * H + o] = im_tanh(acc[r]);
        }
        __syncwarp();
        for (uint32_t o = lane; o < NO; o += 32) {
            float acc[kF32RowsPerWarp];
#pragma unroll
            for (int r = 0; r < kF32RowsPerWarp; r++) acc[r] = sb3[o];
            for (uint32_t k = 0; k < H; k++) {
                const float w = sW3[k * NOP + o];
#pragma unroll
                for (int r = 0; r < kF32RowsPerWarp; r++) acc[r] = __fmaf_rn(w, h2[r * H + k], acc[r]);
            }
#pragma unroll
            for (int r = 0; r < kF32RowsPerWarp; r++) lg[r * 64 + o] = acc[r];
        }
        __syncwarp();
        if (lane < kF32RowsPerWarp) {
            // lane r finishes row r
            bool mine = false; RowInfo mi = ri[0];
#pragma unroll
            for (int r = 0; r < kF32RowsPerWarp; r++) if (lane == (uint32_t)r) { mine = ok[r]; mi = ri[r]; }
            if (mine) {
                if (EXEC) exec_epilogue(P, mi, lg + lane * 64, scr + lane * 64, t0, trow);
                else plan_epilogue(P, mi, lg + lane * 64, scr + lane * 64, t0);
            }
        }
        __syncwarp();
    }
}

size_t f32_smem_bytes(uint32_t F, uint32_t H, uint32_t NOP)
{
    return 4ull * (F * H + H * H + H * NOP + 2 * H + NOP + kF32Warps * kF32RowsPerWarp * (F + 2 * H + 128));
}

// ================================================================================================ tcgen05 path (R25)
// F = 128, H = 256 (configs 4-5): a real dense GEMM, so it runs on the 5th-generation tensor cores (im_tc.cuh).
// One persistent CTA per SM; the whole net (192 KB of bf16 weights) stays in shared memory for the lifetime of the
// launch; a tile is 128 rows = 128 TMEM lanes = 128 threads, thread r owning row r from feature gather to sampling.
// Layer 1 contracts only the first 64 features: rows are zero beyond 3N + 12 <= 60 (R15), so this is exact.
constexpr int kTcK1 = 64, kTcH = 256, kTcThreads = 256;
template <bool EXEC> using TcNet = tc::TcMlp<kTcK1, kTcH, EXEC ? 64 : 32>;

// The tcgen05 kernel is built for K1 = 64 contracted features (any f_in >= 3N + 13) and a hidden width of 256; a net with
// hidden = 128 runs on it zero-padded (k_pack_tc): the padded units have zero weights and biases, tanh(0) = 0, so they add
// exactly nothing - and the kernel skips them: only the first N-half of the hidden layers and half of the K-steps of layers 2
// and 3 are issued, only the first half of the tanh epilogues runs (`narrow`).
bool tc_supported(uint32_t F, uint32_t H) { return (F == 64 && H == 128) || (F == 128 && H == 256); }
size_t tc_image_bytes(bool exec) { return exec ? TcNet<true>::kImageBytes : TcNet<false>::kImageBytes; }

// K order of layer 1 on this path: [snap(3N) | b | in_tok | topo(4) | role(4) | agent | keff | 0...] — the R15 features with
// the budget feature moved behind the snapshot block, so that a row's snapshot floats land on 16-byte chunk boundaries.
// fp32 accumulation order is unspecified under R25, so permuting k is free; W1's columns are permuted to match.
__device__ __forceinline__ uint32_t tc_feature_src(uint32_t kp, uint32_t N3) { return kp < N3 ? kp + 1u : (kp == N3 ? 0u : kp); }

// bf16 [o][k] row-major weights + fp32 biases (k_repack's output) -> the shared-memory image of im_tc.cuh
template <bool EXEC>
__global__ void k_pack_tc(const Weights W, uint32_t N3, uint32_t F, uint32_t H)        // F, H: the net's own f_in and hidden (<= 128, <= 256)
{
    using Net = TcNet<EXEC>;
    constexpr uint32_t NO = EXEC ? 64 : 32;
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
    const __nv_bfloat16 zero = __float2bfloat16(0.0f);
    uint8_t *img = W.tc_img;
    for (uint32_t i = tid; i < kTcH * kTcK1; i += nth) {
        const uint32_t o = i / kTcK1, kp = i % kTcK1, src = tc_feature_src(kp, N3);
        *reinterpret_cast<__nv_bfloat16 *>(img + Net::kW1 + tc::canon_off(kTcH, o, kp)) = (o < H && src < F) ? W.W1[o * F + src] : zero;
    }
    for (uint32_t i = tid; i < kTcH * kTcH; i += nth) {
        const uint32_t o = i / kTcH, k = i % kTcH;
        *reinterpret_cast<__nv_bfloat16 *>(img + Net::kW2 + tc::canon_off(kTcH, o, k)) = (o < H && k < H) ? W.W2[o * H + k] : zero;
    }
    for (uint32_t i = tid; i < NO * kTcH; i += nth) {
        const uint32_t o = i / kTcH, k = i % kTcH;
        *reinterpret_cast<__nv_bfloat16 *>(img + Net::kW3 + tc::canon_off(NO, o, k)) = (o < W.n_out_pad && k < H) ? W.W3[o * H + k] : zero;
    }
    float *bias = reinterpret_cast<float *>(img + Net::kBias);
    for (uint32_t i = tid; i < kTcH; i += nth) { bias[i] = i < H ? W.b1[i] : 0.0f; bias[kTcH + i] = i < H ? W.b2[i] : 0.0f; }
    for (uint32_t i = tid; i < NO; i += nth) bias[2 * kTcH + i] = i < W.n_out_pad ? W.b3[i] : 0.0f;
}

void launch_pack_tc(const Weights &W, bool exec, uint32_t n_models, uint32_t f_in, uint32_t hidden, cudaStream_t st)
{
    if (exec) k_pack_tc<true><<<64, 256, 0, st>>>(W, 3 * n_models, f_in, hidden);
    else k_pack_tc<false><<<64, 256, 0, st>>>(W, 3 * n_models, f_in, hidden);
}

// R24 sampler on logits held in registers: l[off .. off+n), n <= NMAX.  Same VALUES as sample_seq, arranged for a lone
// warp, which pays ~5 cycles per instruction here (profiles/r1_ncu_final_cfg5.md): logits beyond n become -inf (their
// exponential is exactly 0, so the running sums simply stop growing); the max is a tree (exact); the sums
// c_i = c_{i-1} + e_i are computed once in ascending order (Z is the last); since they never decrease, the first i
// with c_i > u Z is the NUMBER of i with c_i <= u Z (capped at n - 1).
template <int NMAX, int NO>
__device__ __forceinline__ uint32_t sample_reg(const float (&l)[NO], int off, uint32_t n, float u, float &logp)
{
    float c[NMAX], mx[NMAX];
#pragma unroll
    for (int i = 0; i < NMAX; i++) { c[i] = (uint32_t)i < n ? l[off + i] : -INFINITY; mx[i] = c[i]; }
#pragma unroll
    for (int s = 1; s < NMAX; s <<= 1)
#pragma unroll
        for (int i = 0; i + s < NMAX; i += 2 * s) mx[i] = fmaxf(mx[i], mx[i + s]);
    const float m = mx[0];
    static_assert(NMAX % 2 == 0, "pairs");
#pragma unroll
    for (int i = 0; i < NMAX; i += 2) im_exp_x2(__fsub_rn(c[i], m), __fsub_rn(c[i + 1], m), c[i], c[i + 1]);
#pragma unroll
    for (int i = 1; i < NMAX; i++) c[i] = __fadd_rn(c[i - 1], c[i]);          // c_0 = 0 + e_0 = e_0
    const float Z = c[NMAX - 1];
    const float th = __fmul_rn(u, Z);
    uint32_t cnt = 0;
#pragma unroll
    for (int i = 0; i < NMAX; i++) cnt += c[i] <= th ? 1u : 0u;
    const uint32_t a = min(cnt, n - 1u);
    float la = l[off];
#pragma unroll
    for (int i = 1; i < NMAX; i++) la = (uint32_t)i == a ? l[off + i] : la;
    logp = __fsub_rn(__fsub_rn(la, m), logf(Z));
    return a;
}

struct TcRaw { uint4 row; uint32_t env, gidx; bool ok, critic; };

// Loads of the NEXT tile's inputs are issued one tile ahead of their use; `asm volatile` keeps ptxas from sinking them
// to the point of use (measured: the feature build then waits two dependent round trips, 1.5 us per tile).
__device__ __forceinline__ uint4 ld_early_u4(const uint4 *p)
{
    uint4 v;
    asm volatile("ld.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ float4 ld_early_f4(const float4 *p)
{
    float4 v;
    asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p) : "memory");
    return v;
}

// row `r` of tile `tile`: issues the row load, decodes nothing (the consumer decodes after the latency has passed)
__device__ __forceinline__ TcRaw tc_fetch_row(const TileSched &S, const RowBuf &rb, uint32_t tile, uint32_t r, uint32_t n_crit)
{
    TcRaw x;
    x.env = 0; x.gidx = 0; x.ok = false; x.critic = false;
    if (tile < S.total) {
        if (tile < S.crit_tiles) {
            const uint32_t env = tile * 128u + r;
            x.ok = env < n_crit; x.critic = true; x.env = env;
        } else {
            const uint32_t lt = tile - S.crit_tiles;
            uint32_t lo = 0, hi = kRegions;
            while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if (S.pref[mid] <= lt) lo = mid; else hi = mid; }
            const uint32_t off = (lt - S.pref[lo]) * 128u + r;
            if (S.base[lo] + off < S.cnt[lo]) {
                uint32_t pos = S.base_mod[lo] + off;             // off < cnt - base <= regcap (checked by sched_init): one wrap at most
                if (pos >= rb.regcap) pos -= rb.regcap;
                x.gidx = lo * rb.regcap + pos;
                x.ok = true;
            }
        }
    }
    // ONE unconditional load on the single exit path (row 0 of the list for a row that does not exist or a critic row: never
    // decoded): a load under a condition is merged by a select, and the select waits for the load
    x.row = ld_early_u4(rb.row + x.gidx);
    return x;
}

template <bool EXEC>
__device__ __forceinline__ RowInfo tc_decode_row(const Params &P, const TcRaw &x, int32_t t0)
{
    RowInfo ri;
    ri.critic = x.critic; ri.gidx = x.gidx;
    if (x.critic) { ri.env = x.env; ri.a = 0; ri.c = 0; ri.dl = 0; ri.b = 0.0f; return ri; }
    ri.env = x.row.x; ri.a = x.row.y; ri.dl = (int32_t)x.row.z; ri.c = x.row.w;
    const int32_t t = t0 + (int32_t)(x.row.y >> 19);
    float b = __fdiv_rn(__int2float_rn(ri.dl - t), __uint2float_rn(P.budget_norm));
    if (EXEC) b = fminf(fmaxf(b, -1.0f), 1.0f);
    ri.b = b;
    return ri;
}

// Row handed from the gathering warpgroup to the sampling warpgroup through shared memory
struct TcRowSlot { uint4 row; uint32_t env, gidx, flags, pad; };           // flags: bit 0 ok, bit 1 critic

template <bool EXEC, bool NARROW>
__global__ void __launch_bounds__(kTcThreads, 1)
k_policy_tc(const Params P, const Weights W, uint32_t parity, int32_t t0, uint32_t trow)
{
    using Net = TcNet<EXEC>;
    constexpr int NO = EXEC ? 64 : 32;
    extern __shared__ __align__(1024) uint8_t smem_tc[];
    __shared__ TileSched sched;
    __shared__ uint64_t bars[5];                          // layer 1 half a / b, layer 2 half a / b, layer 3
    __shared__ uint64_t wbar;                             // arrival of the weight image
    __shared__ uint32_t tmem_slot;
    uint8_t *img = smem_tc, *a1 = smem_tc + ((Net::kImageBytes + 1023u) & ~1023u);
    TcRowSlot *rowbuf = reinterpret_cast<TcRowSlot *>(a1 + Net::kA1Bytes);     // [2][128]
    // the weight image (194 KB) comes by bulk async copies (TMA): one thread issues them, they fly while the CTA allocates
    // its tensor memory, builds the tile schedule and gathers its first tile; everybody waits on wbar before the first use
    if (threadIdx.x == 0) {
        for (int i = 0; i < 5; i++) tc::mbar_init(&bars[i], 1);
        tc::mbar_init(&wbar, 1);
        tc::mbar_fence_init();
        bulk::mbar_expect_tx(&wbar, Net::kImageBytes);
        constexpr uint32_t kPiece = 48 * 1024;
        for (uint32_t o = 0; o < Net::kImageBytes; o += kPiece)
            bulk::g2s(img + o, W.tc_img + o, Net::kImageBytes - o < kPiece ? Net::kImageBytes - o : kPiece, &wbar);
    }
    if (threadIdx.x < 32) tc::tmem_alloc(&tmem_slot, Net::kTmemCols);
    griddep_wait();                                       // the weights were packed before the rollout's first kernel; the rows are the predecessor's
    const RowBuf &rb = EXEC ? P.exec : P.plan;
    const uint32_t n_crit = EXEC ? P.E : 0u;
    sched_init(P, sched, rb, parity, 128, n_crit);
    tc::tc_fence_before();
    __syncthreads();
    tc::tc_fence_after();
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, tmem_slot, 0);          // (the shuffles tell ptxas that these are warp-uniform:
    const uint32_t warp_u = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);      //  the UMMA operands then live in uniform registers)
    const uint32_t N3 = 3 * P.N;
    const bool vec = (N3 % 8u) == 0;                      // snapshot block = whole 16-byte chunks (N = 8, 16)
    constexpr bool narrow = NARROW;                       // a 128-wide net on the 256-wide kernel: half a of the hidden layers only
    const uint32_t wg = warp_u >> 2, r = threadIdx.x & 127u;
    const uint32_t tlane = tmem_base + (((threadIdx.x >> 5) & 3u) * 32u << 16);
    const float *bias = reinterpret_cast<const float *>(img + Net::kBias);
    const uint32_t total = sched.total;
    uint32_t phase = 0, it = 0;                           // mbarrier parity and tile counter of this CTA

    // snapshot floats of a row's env (R14): up to 12 float4 per thread, issued early, consumed one tile later
    auto fetch_snap = [&](const TcRaw &x, float4 (&sn)[12]) {
        // Unconditional loads from an address that is always valid (env 0 for a padding row, chunk 0 beyond 3N): a load
        // under a condition ends in a select, and the select waits for the load - 2000 cycles of DRAM latency per tile that
        // were meant to pass behind the tanh epilogue.  build_a1 reads only the chunks below 3N, and only of rows that exist.
        const uint32_t env = (x.ok && vec) ? (x.critic ? x.env : x.row.x) : 0u;
        const float4 *src = reinterpret_cast<const float4 *>(P.snap + (size_t)env * N3);
#pragma unroll
        for (int j = 0; j < 12; j++) sn[j] = ld_early_f4(src + ((uint32_t)(4 * j) < N3 ? j : 0));
    };
    // features of row `cur` -> A1 (bf16 RNE), canonical layout: chunk c of row r at c * 2048 + r * 16; row -> rowbuf
    auto build_a1 = [&](const TcRaw &cur, const float4 (&sn)[12], TcRowSlot *slot) {
        const RowInfo ri = tc_decode_row<EXEC>(P, cur, t0);
        const bool ok = cur.ok;
        slot[r].row = cur.row; slot[r].env = cur.env; slot[r].gidx = cur.gidx; slot[r].flags = (ok ? 1u : 0u) | (cur.critic ? 2u : 0u);
        if (vec) {
            float tl[16];                                 // the 12 features behind the snapshot block (R15), then zeros
#pragma unroll
            for (int j = 0; j < 16; j++) tl[j] = 0.0f;
            if (ok) {
                tl[0] = ri.b;
                if (!ri.critic) {
                    tl[1] = __uint2float_rn(ri.c & 0xFFFFu) * 0x1p-13f;
                    if (EXEC) {
                        const uint32_t topo = (ri.a >> 12) & 3u, role = (ri.a >> 14) & 3u;
#pragma unroll
                        for (int j = 0; j < 4; j++) { tl[2 + j] = (uint32_t)j == topo ? 1.0f : 0.0f; tl[6 + j] = (uint32_t)j == role ? 1.0f : 0.0f; }
                        tl[10] = __uint2float_rn((ri.a >> 10) & 3u) * 0.25f;
                        tl[11] = __uint2float_rn((ri.a >> 16) & 7u) * 0.25f;
                    }
                }
            }
            const uint32_t c0 = N3 / 8;
#pragma unroll
            for (int c = 0; c < kTcK1 / 8; c++) {
                float f[8];
                if ((uint32_t)c < c0) {
                    f[0] = sn[2 * c].x; f[1] = sn[2 * c].y; f[2] = sn[2 * c].z; f[3] = sn[2 * c].w;
                    f[4] = sn[2 * c + 1].x; f[5] = sn[2 * c + 1].y; f[6] = sn[2 * c + 1].z; f[7] = sn[2 * c + 1].w;
                } else {
#pragma unroll
                    for (int j = 0; j < 8; j++) f[j] = (uint32_t)c == c0 ? tl[j] : ((uint32_t)c == c0 + 1 ? tl[8 + j] : 0.0f);
                }
                *reinterpret_cast<uint4 *>(a1 + c * (128 * 16) + r * 16) =
                    make_uint4(tc::pack_bf16(f[0], f[1]), tc::pack_bf16(f[2], f[3]), tc::pack_bf16(f[4], f[5]), tc::pack_bf16(f[6], f[7]));
            }
        } else {
#pragma unroll 1
            for (int c = 0; c < kTcK1 / 8; c++) {
                float f[8];
#pragma unroll
                for (int j = 0; j < 8; j++) f[j] = ok ? feature(P, EXEC, ri, tc_feature_src(8 * c + j, N3)) : 0.0f;
                *reinterpret_cast<uint4 *>(a1 + c * (128 * 16) + r * 16) =
                    make_uint4(tc::pack_bf16(f[0], f[1]), tc::pack_bf16(f[2], f[3]), tc::pack_bf16(f[4], f[5]), tc::pack_bf16(f[6], f[7]));
            }
        }
    };
    // ---- prologue: warpgroup 1 gathers the first tile and starts its layer 1
    // Row prefetch runs TWO tiles ahead of the tile whose layer 1 is being read out, the snapshot of its env one tile ahead:
    // the snapshot address comes out of the row, so a row fetched only one tile ahead put a full DRAM round trip (2000+
    // cycles under load) into warpgroup 1's serial path on every tile of executor rows.
    TcRaw nxt, nxt2;
    float4 sn[12];
    if (wg == 1) {
        nxt = tc_fetch_row(sched, rb, blockIdx.x, r, n_crit);
        fetch_snap(nxt, sn);
        if (blockIdx.x < total) {
            build_a1(nxt, sn, rowbuf);
            tc::fence_proxy_async_smem();
            tc::bar_sync(4, 128);
            tc::mbar_wait(&wbar, 0);
            if (warp_u == 4) Net::issue_l1(img, a1, tmem_base, &bars[0], &bars[1], narrow);
            nxt = tc_fetch_row(sched, rb, blockIdx.x + gridDim.x, r, n_crit);
            fetch_snap(nxt, sn);
            nxt2 = tc_fetch_row(sched, rb, blockIdx.x + 2 * gridDim.x, r, n_crit);
        }
    }
    tc::mbar_wait(&wbar, 0);
    // One loop per warpgroup.  (With one loop and a branch on the warpgroup inside it, the loop's back edge is a merge of
    // both roles and ptxas waits there for EVERY outstanding scoreboard: warpgroup 1 sat out the 2000 cycles of its
    // snapshot prefetch at the top of every tile instead of behind the tanh epilogue.)
    if (wg == 1) {
        for (uint32_t tile = blockIdx.x; tile < total; tile += gridDim.x, it++, phase ^= 1u) {
            // ---- warpgroup 1: tanh of layer 1, packed in place (half a while the tensor core computes half b)
            tc::mbar_wait(&bars[0], phase);
            tc::tc_fence_after();
            Net::half_epilogue(tlane, 0, 0, bias);
            if (!narrow) {
                tc::mbar_wait(&bars[1], phase);
                tc::tc_fence_after();
                Net::half_epilogue(tlane, 128, 64, bias + 128);
            }
            tc::tc_fence_before();
            tc::bar_sync(2, 128);
            // layer 2 overwrites D3 / A3 of the previous tile: wait until warpgroup 0 has its logits in registers
            if (it > 0) tc::bar_sync(3, 256);
            if (warp_u == 4) Net::issue_l2(img, tmem_base, &bars[2], &bars[3], narrow);
            // the next tile: features (layer 1 of this tile is done with a1), layer 1 behind layer 2 in the tensor pipe
            // (UMMAs of one thread execute in order, so A2 is consumed by then), row loads of the tile after it
            if (tile + gridDim.x < total) {
                build_a1(nxt, sn, rowbuf + 128 * ((it + 1) & 1u));
                tc::fence_proxy_async_smem();
                tc::bar_sync(4, 128);
                if (warp_u == 4) Net::issue_l1(img, a1, tmem_base, &bars[0], &bars[1], narrow);
                nxt = nxt2;                                   // row of tile + 2 grids: its load went out one tile ago
                fetch_snap(nxt, sn);
                nxt2 = tc_fetch_row(sched, rb, tile + 3 * gridDim.x, r, n_crit);
            }
        }
    } else
    for (uint32_t tile = blockIdx.x; tile < total; tile += gridDim.x, it++, phase ^= 1u) {
        // ---- warpgroup 0: tanh of layer 2, packed in place (half a while the tensor core computes half b), layer 3
        tc::mbar_wait(&bars[2], phase);
        tc::tc_fence_after();
        Net::half_epilogue(tlane, Net::kColD2, Net::kColD2, bias + kTcH);
        if (!narrow) {
            tc::mbar_wait(&bars[3], phase);
            tc::tc_fence_after();
            Net::half_epilogue(tlane, Net::kColD2 + 128, Net::kColD2 + 128, bias + kTcH + 128);
        }
        tc::tc_fence_before();
        tc::bar_sync(5, 128);
        if (warp_u == 0) Net::issue_l3(img, tmem_base, &bars[4], narrow);
        // ---- warpgroup 0: sampling epilogue of row r, logits in registers
        const TcRowSlot sl = rowbuf[128 * (it & 1u) + r];
        uint32_t islot = ~0u;                              // executor rows: the env's issue-list slot, claimed before the wait
        if (EXEC && (sl.flags & 3u) == 1u) islot = atomicAdd(hdr_word(P, sl.row.x, P.hw_misc + 1u), 1u);
        tc::mbar_wait(&bars[4], phase);
        tc::tc_fence_after();
        float l[NO];
        Net::load_logits(img, tlane, l);
        const float value = EXEC ? Net::load_output(img, tlane, N3) : 0.0f;     // critic / value head (R26: row 3N)
        tc::tc_fence_before();
        if (tile + gridDim.x < total) tc::bar_arrive(3, 256);   // warpgroup 1 may now issue the next tile's layer 2
        const bool ok = (sl.flags & 1u) != 0;
        if (EXEC && !ok) continue;
        TcRaw cur;
        cur.row = sl.row; cur.env = sl.env; cur.gidx = sl.gidx; cur.ok = ok; cur.critic = (sl.flags & 2u) != 0;
        const RowInfo ri = tc_decode_row<EXEC>(P, cur, t0);
        if (EXEC) {
            const uint32_t n = N3;
            if (ri.critic) {
                P.val[(size_t)trow * P.E + ri.env] = value;
            } else {
                if (P.exec.logits) {
#pragma unroll
                    for (int i = 0; i < NO; i++) if ((uint32_t)i <= n) P.exec.logits[(size_t)ri.gidx * P.exec.n_out + i] = l[i];
                }
                const uint32_t q = ri.a & 0x3FFu, agent = (ri.a >> 10) & 3u;
                const int32_t t = t0 + (int32_t)(ri.a >> 19);
                const Ph4 d = draw(P, STREAM_EXEC, P.env_id_base + ri.env, t, q * 4u + agent, 0);
                float logp;
                const uint32_t act = sample_reg<48, NO>(l, 0, n, u24(d.x), logp);
                exec_commit(P, ri, d, act, logp, value, t, islot);
            }
        } else {
            uint32_t topo = 0, cnt = 0, roles = 0, nc = 0;
            float lp = 0.0f;
            if (ok) {
                if (P.plan.logits) {
#pragma unroll
                    for (int i = 0; i < 24; i++) P.plan.logits[(size_t)ri.gidx * 24 + i] = l[i];
                }
                const uint32_t q = ri.a & 0x3FFu;
                const int32_t t = t0 + (int32_t)(ri.a >> 19);
                const uint32_t gid = P.env_id_base + ri.env;
                const Ph4 d0 = draw(P, STREAM_PLAN, gid, t, q, 0), d1 = draw(P, STREAM_PLAN, gid, t, q, 1);
                float lp_t, lp_c, lp_r[4];
                topo = sample_reg<4, NO>(l, 0, 4, u24(d0.x), lp_t);
                cnt = sample_reg<4, NO>(l, 4, 4, u24(d0.y), lp_c);
                const uint32_t ur[4] = {d1.x, d1.y, d1.z, d1.w};
#pragma unroll
                for (int a = 0; a < 4; a++) roles |= sample_reg<4, NO>(l, 8 + 4 * a, 4, u24(ur[a]), lp_r[a]) << (2 * a);
                const uint32_t keff = keff_of(topo, cnt + 1);
                lp = __fadd_rn(lp_t, lp_c);
#pragma unroll
                for (uint32_t a = 0; a < 4; a++) if (a < keff) lp = __fadd_rn(lp, lp_r[a]);
                uint32_t a0;
                stage_calls(topo, keff, 0, a0, nc);
            }
            // one claim per warp: the rows of a tile belong to one region (the tile schedule is per region)
            const uint32_t lane = threadIdx.x & 31u;
            uint32_t inc = nc;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= (uint32_t)o) inc += v; }
            const uint32_t tot = __shfl_sync(0xffffffffu, inc, 31), okm = __ballot_sync(0xffffffffu, ok);
            if (tot) {
                const uint32_t region = __shfl_sync(0xffffffffu, region_of(P, ri.env), __ffs(okm) - 1);
                uint32_t base = 0;
                if (lane == 0) base = rows_claim(P, P.exec, region, tot) % P.exec.regcap;
                uint32_t idx0 = __shfl_sync(0xffffffffu, base, 0) + inc - nc;
                if (idx0 >= P.exec.regcap) idx0 -= P.exec.regcap;
                if (ok) plan_commit(P, ri, topo, cnt, roles, lp, idx0);
            }
        }
    }
    tc::tc_fence_before();
    __syncthreads();
    if (threadIdx.x < 32) tc::tmem_dealloc(tmem_base, Net::kTmemCols);
}

// ------------------------------------------------------------------------------------------------ launchers
// opt-in to large dynamic shared memory on the CURRENT device (the attribute is per device: im_bind calls this once per ctx)
int policy_prepare_device(const Params &P)
{
    const int big = 200 * 1024;
    cudaError_t e = cudaSuccess;
    auto set = [&](const void *f, int bytes) { if (e == cudaSuccess) e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes); };
    set((const void *)k_policy_f32<true>, big);
    set((const void *)k_policy_f32<false>, big);
    const int tc_smem = (int)(((tc_image_bytes(true) + 1023u) & ~(size_t)1023u) + TcNet<true>::kA1Bytes + 2 * 128 * sizeof(TcRowSlot));
    set((const void *)k_policy_tc<true, false>, tc_smem);
    set((const void *)k_policy_tc<false, false>, tc_smem);
    set((const void *)k_policy_tc<true, true>, tc_smem);
    set((const void *)k_policy_tc<false, true>, tc_smem);
    (void)P;
    return e == cudaSuccess ? 0 : -1;
}

int launch_policy(const Params &P, const Weights &W, bool exec, uint32_t parity, int32_t t0, uint32_t trow, int n_sm,
                  bool bf16, cudaStream_t st)
{
    if (!bf16) {
        const size_t smem = f32_smem_bytes(P.f_in, P.hidden, W.n_out_pad);
        const uint32_t grid = (uint32_t)n_sm * 2;
        if (exec) k_policy_f32<true><<<grid, kF32Warps * 32, smem, st>>>(P, W, parity, t0, trow);
        else k_policy_f32<false><<<grid, kF32Warps * 32, smem, st>>>(P, W, parity, t0, trow);
        return 0;
    }
    if (W.tc_img) {      // bf16: tcgen05 (hidden = 128 zero-padded to 256, k_pack_tc)
        const size_t smem = ((tc_image_bytes(exec) + 1023u) & ~(size_t)1023u) + TcNet<true>::kA1Bytes + 2 * 128 * sizeof(TcRowSlot);
        const bool narrow = P.hidden <= 128;             // template parameter: the wide kernel compiles without a trace of it
        if (exec) {
            if (narrow) launch_chained(k_policy_tc<true, true>, dim3(n_sm), dim3(kTcThreads), smem, st, true, P, W, parity, t0, trow);
            else launch_chained(k_policy_tc<true, false>, dim3(n_sm), dim3(kTcThreads), smem, st, true, P, W, parity, t0, trow);
        } else {
            if (narrow) launch_chained(k_policy_tc<false, true>, dim3(n_sm), dim3(kTcThreads), smem, st, true, P, W, parity, t0, trow);
            else launch_chained(k_policy_tc<false, false>, dim3(n_sm), dim3(kTcThreads), smem, st, true, P, W, parity, t0, trow);
        }
        return 0;
    }
    return -1;
}

}  // namespace im
