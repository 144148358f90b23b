// im_sim.cu — the fixed-tick simulation kernel: one warp per environment.
//
// One launch runs, for every env, the environment half of the canonical tick:
//   post(t):  D-issue (requests of the decisions k_exec took for tick t), E admit (slack-ordered queue, R20/R21),
//             F serve (token-level service, R11), G complete (latency, cost, EWMA, finalise, R13/R27/R28),
//             H preempt (R21), I record (R27/R28/R33)
//   pre(t+1): A arrive (Poisson count, budgets, input tokens; R5-R9), B snapshot (R14), and the emission of the
//             work lists: one planner row per new query, executor rows for every query whose previous stage
//             completed (R17).
// The decision half (C plan, D decide) runs between two launches in im_policy.cu.
//
// Layout: SoA arrays [E][cap] with the cap index fastest, so a warp streams one env's field with 128-bit loads
// (north_star (1)).  Everything order-dependent in the definition (j-th new item takes the j-th lowest free index,
// R9/R18) is done by ranked selection on free bitmaps; every accumulation is an integer sum, so lanes may commit
// in any order (R12, R13, R28).
#include "im_device.cuh"

namespace im {

constexpr int kSimWarps = 8;

struct WarpSmem {
    uint32_t *rfree;     // [RW] free bitmap at kernel start (lookups)
    uint32_t *rfree_new; // [RW] free bitmap being updated
    uint32_t *qfree;     // [QW]
    uint32_t *qready;    // [QW]
    uint32_t *prefA;     // [RW+1]
    uint32_t *prefB;     // [QW+1]
    uint32_t *mc;        // [6][16] n_wait, n_run, kv_used, ewma, lat_sum, lat_n
    unsigned long long *cand; // [RCAP]
};

__host__ __device__ inline size_t sim_warp_smem_bytes(uint32_t RCAP, uint32_t QCAP)
{
    const uint32_t RW = RCAP / 32, QW = QCAP / 32;
    size_t words = 2 * RW + 2 * QW + (RW + 1) + (QW + 1) + 6 * 16;
    words = (words + 1) & ~(size_t)1;
    return words * 4 + (size_t)RCAP * 8;
}

__device__ __forceinline__ uint32_t warp_sum(uint32_t v)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, uint32_t lane)
{
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t n = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= (uint32_t)o) v += n;
    }
    return v;
}

// exclusive prefix of popcounts of bm[0..nw) into pref[0..nw]; returns the total
__device__ __forceinline__ uint32_t build_prefix(const uint32_t *bm, uint32_t nw, uint32_t *pref, uint32_t lane)
{
    uint32_t carry = 0;
    for (uint32_t w0 = 0; w0 < nw; w0 += 32) {
        const uint32_t w = w0 + lane;
        const uint32_t pc = w < nw ? __popc(bm[w]) : 0u;
        const uint32_t inc = warp_incl_scan(pc, lane);
        if (w < nw) pref[w] = carry + inc - pc;
        carry += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) pref[nw] = carry;
    __syncwarp();
    return carry;
}

// index of the j-th (0-based) set bit of bm, given its exclusive popcount prefix
__device__ __forceinline__ uint32_t find_nth(const uint32_t *bm, uint32_t nw, const uint32_t *pref, uint32_t j)
{
    uint32_t lo = 0, hi = nw;         // invariant: pref[lo] <= j < pref[hi]
    while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (pref[mid] <= j) lo = mid; else hi = mid;
    }
    return lo * 32 + __fns(bm[lo], 0, (int)(j - pref[lo]) + 1);
}

__device__ __forceinline__ uint32_t queue_key(const Params &P, int32_t deadline, int32_t issue, uint32_t ridx, int32_t t)
{
    const int32_t base = P.sched_mode ? deadline : issue;
    return ((uint32_t)(base - t + (1 << 19)) << 12) | ridx;
}

// tick arguments: t_post < 0 => no post phases; pre_mode 0 none, 1 full (A, B, rows), 2 snapshot only
__global__ void __launch_bounds__(kSimWarps * 32)
k_sim(const Params P, int32_t t_post, uint32_t trow_post, int32_t t_pre, uint32_t pre_mode, int32_t t0)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ ModelTab s_model[kMaxModels];
    const uint32_t lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    if (threadIdx.x < P.N) s_model[threadIdx.x] = P.model[threadIdx.x];
    __syncthreads();
    const uint32_t e = blockIdx.x * kSimWarps + wib;
    if (e >= P.E) return;
    const uint32_t gid = P.env_id_base + e;
    const uint32_t N = P.N, RW = P.RW, QW = P.QW, RCAP = P.RCAP, QCAP = P.QCAP;
    const uint32_t region = e % kRegions;

    WarpSmem S;
    {
        unsigned char *base = smem_raw + (size_t)wib * sim_warp_smem_bytes(RCAP, QCAP);
        S.cand = (unsigned long long *)base;
        uint32_t *w = (uint32_t *)(base + (size_t)RCAP * 8);
        S.rfree = w; w += RW;
        S.rfree_new = w; w += RW;
        S.qfree = w; w += QW;
        S.qready = w; w += QW;
        S.prefA = w; w += RW + 1;
        S.prefB = w; w += QW + 1;
        S.mc = w;
    }
    uint32_t *s_nwait = S.mc, *s_nrun = S.mc + 16, *s_kv = S.mc + 32, *s_ewma = S.mc + 48, *s_latsum = S.mc + 64, *s_latn = S.mc + 80;

    uint32_t *r_meta = P.r_meta + (size_t)e * RCAP, *r_rs = P.r_rs + (size_t)e * RCAP, *r_tok = P.r_tok + (size_t)e * RCAP;
    int32_t *r_dl = P.r_dl + (size_t)e * RCAP, *r_issue = P.r_issue + (size_t)e * RCAP;
    uint32_t *q_plan = P.q_plan + (size_t)e * QCAP, *q_bi = P.q_bi + (size_t)e * QCAP, *q_row = P.q_row + (size_t)e * QCAP;
    int32_t *q_dl = P.q_dl + (size_t)e * QCAP, *q_arr = P.q_arr + (size_t)e * QCAP;

    // ---- load per-env small state
    for (uint32_t w = lane; w < RW; w += 32) { const uint32_t v = P.r_free[(size_t)e * RW + w]; S.rfree[w] = v; S.rfree_new[w] = v; }
    for (uint32_t w = lane; w < QW; w += 32) { S.qfree[w] = P.q_free[(size_t)e * QW + w]; S.qready[w] = P.q_ready[(size_t)e * QW + w]; }
    if (lane < 16) {
        uint4 m = make_uint4(0, 0, 0, 0);
        if (lane < N) m = P.m_cnt[(size_t)e * N + lane];
        s_nwait[lane] = m.x; s_nrun[lane] = m.y; s_kv[lane] = m.z; s_ewma[lane] = m.w; s_latsum[lane] = 0; s_latn[lane] = 0;
    }
    __syncwarp();

    // lane-local counter contributions, merged at the end (lane i adds into counter i after a warp reduction)
    uint32_t c_finished = 0, c_solved = 0, c_missed = 0, c_issued = 0, c_done = 0, c_preempt = 0, c_sojourn = 0;
    uint32_t c_arrivals = 0, c_dropped = 0, c_plans = 0, c_live_mid = 0, c_running = 0, c_waiting = 0, c_abandoned = 0;

    if (t_post >= 0) {
        const int32_t t = t_post;
        // =============================================================== D-issue (R18): canonical request indices
        {
            const uint32_t n_ready = build_prefix(S.qready, QW, S.prefB, lane);
            if (n_ready) {
                build_prefix(S.rfree, RW, S.prefA, lane);
                uint32_t rank0 = 0;
                for (uint32_t b0 = 0; b0 < n_ready; b0 += 32) {
                    const uint32_t o = b0 + lane;
                    uint32_t q = 0, pw = 0, a0 = 0, nc = 0;
                    if (o < n_ready) {
                        q = find_nth(S.qready, QW, S.prefB, o);
                        pw = __ldcg(&q_plan[q]);
                        stage_calls((pw >> 2) & 3, (pw >> 6) & 7, (pw >> 9) & 7, a0, nc);
                    }
                    const uint32_t inc = warp_incl_scan(nc, lane);
                    uint32_t rank = rank0 + inc - nc;
                    rank0 += __shfl_sync(0xffffffffu, inc, 31);
                    if (o < n_ready) {
                        const uint32_t bi = q_bi[q];
                        const uint32_t in_tok = bi >> 16;
                        const int32_t dl = q_dl[q];
                        const uint32_t row0 = q_row[q];
                        for (uint32_t j = 0; j < nc; j++, rank++) {
                            const uint32_t agent = a0 + j;
                            const uint32_t ridx = find_nth(S.rfree, RW, S.prefA, rank);
                            const uint32_t act = (P.exec.c[row_gid(P.exec, region, row0 + j)] >> 16) & 0xFFu;
                            const uint32_t model = act / 3u, depth = act - model * 3u;
                            const Ph4 d = draw(P, STREAM_EXEC, gid, t, q * 4u + agent, 0);
                            uint32_t out_total = (uint32_t)(((unsigned long long)P.depth_median[depth] * P.tab_mult[d.y >> 22]) >> 16);
                            out_total = out_total < 1u ? 1u : out_total;
                            const uint32_t succ = d.z < s_model[model].succ[depth] ? 1u : 0u;
                            r_meta[ridx] = ST_WAIT | (model << 2) | (depth << 6) | (agent << 8) | (succ << 10) | (q << 16);
                            r_rs[ridx] = out_total;
                            r_tok[ridx] = out_total | (in_tok << 16);
                            r_dl[ridx] = dl;
                            r_issue[ridx] = t;
                            atomicAnd(&S.rfree_new[ridx >> 5], ~(1u << (ridx & 31)));
                            atomicAdd(&s_nwait[model], 1u);
                        }
                        // stage++, pending = nc
                        pw = (pw & ~((7u << 9) | (3u << QP_PEND_SHIFT))) | ((((pw >> 9) & 7) + 1) << 9) | (nc << QP_PEND_SHIFT);
                        q_plan[q] = pw;
                        c_issued += nc;
                    }
                }
                __syncwarp();
                for (uint32_t w = lane; w < QW; w += 32) S.qready[w] = 0;
                __syncwarp();
            }
        }
        // high-water mark of the request pool (highest occupied index + 1)
        uint32_t hwm = 0;
        for (uint32_t w = lane; w < RW; w += 32) {
            const uint32_t occ = ~S.rfree_new[w];
            if (occ) hwm = max(hwm, w * 32 + 32 - __clz(occ));
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) hwm = max(hwm, __shfl_xor_sync(0xffffffffu, hwm, o));
        const uint32_t n_chunks = (hwm + 127) / 128;

        // =============================================================== E admit (R20, R21)
        {
            const bool adm = lane < N && s_nwait[lane] > 0 && s_nrun[lane] < s_model[lane].slots && s_kv[lane] <= s_model[lane].kv_cap;
            const uint32_t madm = __ballot_sync(0xffffffffu, adm);
            if (madm) {
                // stage the WAITING requests of admitting models: (model << 32 | key) in shared memory
                uint32_t n_cand = 0;
                for (uint32_t c = 0; c < n_chunks; c++) {
                    const uint32_t i0 = c * 128 + lane * 4;
                    const uint4 m4 = *reinterpret_cast<const uint4 *>(r_meta + i0);
                    const uint32_t mm[4] = {m4.x, m4.y, m4.z, m4.w};
#pragma unroll
                    for (int s = 0; s < 4; s++) {
                        const uint32_t m = mm[s];
                        const bool is = (m & 3u) == ST_WAIT && ((madm >> ((m >> 2) & 15u)) & 1u);
                        const uint32_t bal = __ballot_sync(0xffffffffu, is);
                        if (is) {
                            const uint32_t i = i0 + s;
                            const uint32_t key = queue_key(P, r_dl[i], r_issue[i], i, t);
                            S.cand[n_cand + __popc(bal & ((1u << lane) - 1u))] = ((unsigned long long)((m >> 2) & 15u) << 32) | key;
                        }
                        n_cand += __popc(bal);
                    }
                }
                __syncwarp();
                // per admitting model: repeated extraction of the smallest key; stop at the first that does not fit
                uint32_t mleft = madm;
                while (mleft) {
                    const uint32_t k = __ffs(mleft) - 1;
                    mleft &= mleft - 1;
                    for (;;) {
                        if (s_nwait[k] == 0 || s_nrun[k] >= s_model[k].slots) break;
                        unsigned long long best = ~0ull; uint32_t bpos = 0;
                        for (uint32_t j = lane; j < n_cand; j += 32) {
                            const unsigned long long v = S.cand[j];
                            if ((uint32_t)(v >> 32) == k && v < best) { best = v; bpos = j; }
                        }
#pragma unroll
                        for (int o = 16; o; o >>= 1) {
                            const unsigned long long ob = __shfl_xor_sync(0xffffffffu, best, o);
                            const uint32_t op = __shfl_xor_sync(0xffffffffu, bpos, o);
                            if (ob < best) { best = ob; bpos = op; }
                        }
                        if (best == ~0ull) break;
                        const uint32_t ridx = (uint32_t)best & 0xFFFu;
                        const uint32_t tk = r_tok[ridx], rs = r_rs[ridx];
                        const uint32_t need = (tk >> 16) + ((tk & 0xFFFFu) - (rs & 0xFFFFu));      // R12
                        if (s_kv[k] + need > s_model[k].kv_cap) break;
                        __syncwarp();
                        if (lane == 0) {
                            r_meta[ridx] = (r_meta[ridx] & ~3u) | ST_RUN;
                            const uint32_t pf = (uint32_t)(((unsigned long long)s_model[k].prefill * need) / 1000u);
                            r_rs[ridx] = (rs & 0xFFFFu) | (pf << 16);
                            S.cand[bpos] = ~0ull;
                            s_kv[k] += need; s_nwait[k] -= 1; s_nrun[k] += 1;
                        }
                        __syncwarp();
                    }
                }
            }
        }
        __syncwarp();

        // =============================================================== F serve (R11) + G complete (R1, R13, R27, R28)
        uint32_t rew_acc = 0, miss_acc = 0;
        unsigned long long cost_acc = 0;
        for (uint32_t c = 0; c < n_chunks; c++) {
            const uint32_t i0 = c * 128 + lane * 4;
            uint4 m4 = *reinterpret_cast<const uint4 *>(r_meta + i0);
            const bool any_run = ((m4.x & 3u) == ST_RUN) | ((m4.y & 3u) == ST_RUN) | ((m4.z & 3u) == ST_RUN) | ((m4.w & 3u) == ST_RUN);
            if (!any_run) continue;
            uint4 rs4 = *reinterpret_cast<const uint4 *>(r_rs + i0);
            const Ph4 u4 = draw(P, STREAM_SVC, gid, t, i0 >> 2, 0);
            uint32_t mm[4] = {m4.x, m4.y, m4.z, m4.w};
            uint32_t rr[4] = {rs4.x, rs4.y, rs4.z, rs4.w};
            const uint32_t uu[4] = {u4.x, u4.y, u4.z, u4.w};
            bool meta_dirty = false;
#pragma unroll
            for (int s = 0; s < 4; s++) {
                const uint32_t m = mm[s];
                if ((m & 3u) != ST_RUN) continue;
                const uint32_t model = (m >> 2) & 15u;
                uint32_t rem = rr[s] & 0xFFFFu, pf = rr[s] >> 16;
                uint32_t usable = kDtUs;
                const uint32_t d = min(pf, usable);
                pf -= d; usable -= d;
                const uint32_t x = s_model[model].rate * usable;
                const uint32_t base = x / 1000000u, frac = x - base * 1000000u;
                const uint32_t extra = __umulhi(uu[s], 1000000u) < frac ? 1u : 0u;
                const uint32_t tok = min(base + extra, rem);
                rem -= tok;
                if (tok) atomicAdd(&s_kv[model], tok);
                rr[s] = rem | (pf << 16);
                if (rem == 0) {
                    // ---- completion of request i
                    const uint32_t i = i0 + s, q = m >> 16;
                    const uint32_t ell = (uint32_t)(t + 1 - r_issue[i]);
                    const uint32_t tk = r_tok[i];
                    const uint32_t budget = q_bi[q] & 0xFFFFu;
                    cost_acc += ((unsigned long long)ell << 16) / budget;            // C_k = l_k / beta, Q16 (R28)
                    atomicAdd(&s_latsum[model], ell);
                    atomicAdd(&s_latn[model], 1u);
                    atomicSub(&s_kv[model], (tk >> 16) + (tk & 0xFFFFu));
                    atomicSub(&s_nrun[model], 1u);
                    c_done++;
                    mm[s] = 0; rr[s] = 0; meta_dirty = true;
                    r_tok[i] = 0; r_dl[i] = 0; r_issue[i] = 0;
                    atomicOr(&S.rfree_new[i >> 5], 1u << (i & 31));
                    const uint32_t delta = (((m >> 10) & 1u) << QP_SUCC_SHIFT) - (1u << QP_PEND_SHIFT);
                    const uint32_t old = atomicAdd(&q_plan[q], delta);
                    if (((old >> QP_PEND_SHIFT) & 3u) == 1u) {
                        const uint32_t nw = old + delta;
                        if (((nw >> 9) & 7u) == ((nw >> 12) & 7u)) {
                            // ---- finalise query q (R27): reward, SLO miss, sojourn, query log
                            const uint32_t solved = ((nw >> QP_SUCC_SHIFT) & 7u) ? 1u : 0u;
                            const int32_t arr = q_arr[q], dl = q_dl[q];
                            const uint32_t sojourn = (uint32_t)(t + 1 - arr);
                            const uint32_t late = (t + 1 > dl) ? 1u : 0u;
                            rew_acc += solved; miss_acc += late;
                            c_finished++; c_solved += solved; c_missed += late; c_sojourn += sojourn;
                            const uint32_t li = atomicAdd(&P.qlog.cnt[region], 1u);
                            if (li >= P.qlog.regcap) atomicOr(P.err_flag, 2u);
                            const uint32_t lg = region * P.qlog.regcap + (li % P.qlog.regcap);
                            P.qlog.env[lg] = gid; P.qlog.arrive[lg] = (uint32_t)arr; P.qlog.sojourn[lg] = sojourn;
                            P.qlog.info[lg] = budget | (solved << 16) | (((nw >> 2) & 3u) << 17) | (((nw >> 6) & 7u) << 19);
                            q_plan[q] = 0; q_bi[q] = 0; q_dl[q] = 0; q_arr[q] = 0;
                            atomicOr(&S.qfree[q >> 5], 1u << (q & 31));
                        } else {
                            atomicOr(&S.qready[q >> 5], 1u << (q & 31));
                        }
                    }
                }
            }
            *reinterpret_cast<uint4 *>(r_rs + i0) = make_uint4(rr[0], rr[1], rr[2], rr[3]);
            if (meta_dirty) *reinterpret_cast<uint4 *>(r_meta + i0) = make_uint4(mm[0], mm[1], mm[2], mm[3]);
        }
        __syncwarp();
        // EWMA latency, one update per model per tick (R13)
        if (lane < N && s_latn[lane] > 0) {
            const int32_t mean_q8 = (int32_t)((s_latsum[lane] << 8) / s_latn[lane]);
            int32_t ew = (int32_t)s_ewma[lane];
            ew += (mean_q8 - ew) >> 3;
            s_ewma[lane] = (uint32_t)ew;
        }
        __syncwarp();

        // =============================================================== H preempt (R21)
        if (P.kv_preempt) {
            const bool over = lane < N && s_kv[lane] > s_model[lane].kv_cap;
            uint32_t mover = __ballot_sync(0xffffffffu, over);
            while (mover) {
                const uint32_t k = __ffs(mover) - 1;
                mover &= mover - 1;
                while (s_kv[k] > s_model[k].kv_cap) {
                    // victim = RUNNING request of model k with the largest (deadline, ridx)
                    long long best = -1;
                    for (uint32_t c = 0; c < n_chunks; c++) {
                        const uint32_t i0 = c * 128 + lane * 4;
                        const uint4 m4 = *reinterpret_cast<const uint4 *>(r_meta + i0);
                        const uint32_t mm[4] = {m4.x, m4.y, m4.z, m4.w};
#pragma unroll
                        for (int s = 0; s < 4; s++)
                            if ((mm[s] & 3u) == ST_RUN && ((mm[s] >> 2) & 15u) == k) {
                                const long long v = (((long long)r_dl[i0 + s] + (1ll << 31)) << 12) | (long long)(i0 + s);
                                best = v > best ? v : best;
                            }
                    }
#pragma unroll
                    for (int o = 16; o; o >>= 1) { const long long ob = __shfl_xor_sync(0xffffffffu, best, o); best = ob > best ? ob : best; }
                    if (best < 0) break;
                    __syncwarp();
                    if (lane == 0) {
                        const uint32_t vi = (uint32_t)(best & 0xFFF);
                        const uint32_t tk = r_tok[vi], rs = r_rs[vi];
                        s_kv[k] -= (tk >> 16) + ((tk & 0xFFFFu) - (rs & 0xFFFFu));
                        r_meta[vi] = (r_meta[vi] & ~3u) | ST_WAIT;
                        r_rs[vi] = rs & 0xFFFFu;
                        s_nrun[k] -= 1; s_nwait[k] += 1;
                        c_preempt++;
                    }
                    __syncwarp();
                }
            }
        }

        // =============================================================== I record (R27, R28, R33)
        {
            rew_acc = warp_sum(rew_acc); miss_acc = warp_sum(miss_acc);
#pragma unroll
            for (int o = 16; o; o >>= 1) cost_acc += __shfl_xor_sync(0xffffffffu, cost_acc, o);
            const uint32_t drops = P.e_hdr[e];                 // R9: drops of this tick's phase A
            miss_acc += drops;
            cost_acc += (unsigned long long)drops << 16;
            const uint32_t done = (P.episode_ticks && ((uint32_t)(t + 1) % P.episode_ticks) == 0) ? 1u : 0u;
            if (lane == 0) {
                const size_t idx = (size_t)trow_post * P.E + e;
                P.rew[idx] = __uint2float_rn(rew_acc);
                P.cost[idx] = P.cost_mode ? __uint2float_rn(miss_acc) : __ull2float_rn(cost_acc) * 0x1p-16f;
                P.miss[idx] = (uint8_t)min(miss_acc, 255u);
                P.done[idx] = (uint8_t)done;
            }
            if (lane < N) { c_running += s_nrun[lane]; c_waiting += s_nwait[lane]; }
            if (done) {
                // hard reset: live queries abandoned, tables emptied
                uint32_t live = 0;
                for (uint32_t w = lane; w < QW; w += 32) live += __popc(~S.qfree[w]);
                c_abandoned += live;
                for (uint32_t i = lane; i < hwm; i += 32) { r_meta[i] = 0; r_rs[i] = 0; r_tok[i] = 0; r_dl[i] = 0; r_issue[i] = 0; }
                for (uint32_t i = lane; i < QCAP; i += 32) { q_plan[i] = 0; q_bi[i] = 0; q_dl[i] = 0; q_arr[i] = 0; }
                for (uint32_t w = lane; w < RW; w += 32) S.rfree_new[w] = 0xFFFFFFFFu;
                for (uint32_t w = lane; w < QW; w += 32) { S.qfree[w] = 0xFFFFFFFFu; S.qready[w] = 0; }
                if (lane < 16) { s_nwait[lane] = 0; s_nrun[lane] = 0; s_kv[lane] = 0; s_ewma[lane] = 0; }
            }
        }
        __syncwarp();
    }

    // ===================================================================== pre(t_pre): A arrive, B snapshot, work lists
    uint32_t drops_next = 0;
    if (pre_mode == 1) {
        const int32_t t = t_pre;
        const uint32_t t_rel = (uint32_t)(t - t0);
        // ---- executor rows of the queries whose previous stage completed (pending == 0, stages left), index ascending
        {
            const uint32_t n_ready = build_prefix(S.qready, QW, S.prefB, lane);
            for (uint32_t b0 = 0; b0 < n_ready; b0 += 32) {
                const uint32_t o = b0 + lane;
                uint32_t q = 0, pw = 0, a0 = 0, nc = 0;
                if (o < n_ready) {
                    q = find_nth(S.qready, QW, S.prefB, o);
                    pw = __ldcg(&q_plan[q]);
                    stage_calls((pw >> 2) & 3, (pw >> 6) & 7, (pw >> 9) & 7, a0, nc);
                }
                const uint32_t inc = warp_incl_scan(nc, lane);
                const uint32_t tot = __shfl_sync(0xffffffffu, inc, 31);
                uint32_t idx0 = 0;
                if (lane == 0 && tot) idx0 = rows_claim(P, P.exec, region, tot);
                idx0 = __shfl_sync(0xffffffffu, idx0, 0) + inc - nc;
                if (o < n_ready) {
                    const uint32_t topo = (pw >> 2) & 3, keff = (pw >> 6) & 7, roles = (pw >> QP_ROLE_SHIFT) & 0xFFu;
                    const uint32_t in_tok = q_bi[q] >> 16;
                    float b = __fdiv_rn(__int2float_rn(q_dl[q] - t), __uint2float_rn(P.budget_norm));
                    b = fminf(fmaxf(b, -1.0f), 1.0f);
                    q_row[q] = idx0;
                    for (uint32_t j = 0; j < nc; j++) {
                        const uint32_t agent = a0 + j, g = row_gid(P.exec, region, idx0 + j);
                        P.exec.env[g] = e;
                        P.exec.a[g] = q | (agent << 10) | (topo << 12) | (((roles >> (2 * agent)) & 3u) << 14) | (keff << 16) | (t_rel << 19);
                        P.exec.b[g] = b;
                        P.exec.c[g] = in_tok;
                    }
                }
            }
        }
        // ---- A arrive (R5, R7, R8, R9)
        {
            const uint32_t xr = draw(P, STREAM_ARR, gid, t, 0, 0).x;
            const uint32_t *cdf = P.tab_cdf + 32u * P.env_level[e];
            const uint32_t n = __popc(__ballot_sync(0xffffffffu, lane < 31 && xr >= cdf[lane]));
            const uint32_t n_free = build_prefix(S.qfree, QW, S.prefB, lane);
            const uint32_t n_ok = min(n, n_free);
            drops_next = n - n_ok;
            c_arrivals += (lane == 0) ? n : 0; c_dropped += (lane == 0) ? drops_next : 0; c_plans += (lane == 0) ? n_ok : 0;
            uint32_t pidx0 = 0;
            if (lane == 0 && n_ok) pidx0 = rows_claim(P, P.plan, region, n_ok);
            pidx0 = __shfl_sync(0xffffffffu, pidx0, 0);
            uint32_t q = 0;
            if (lane < n_ok) {
                q = find_nth(S.qfree, QW, S.prefB, lane);
                const Ph4 d = draw(P, STREAM_QRY, gid, t, lane, 0);
                const uint32_t comp = d.z < P.mix_thresh ? 0u : 1u;
                const uint32_t budget = P.mix_lo[comp] + __umulhi(d.x, P.mix_hi[comp] - P.mix_lo[comp] + 1u);
                const uint32_t in_tok = P.has_intok ? P.tab_intok[d.y >> 22] : P.in_tok_const;
                q_plan[q] = QP_LIVE;
                q_bi[q] = budget | (in_tok << 16);
                q_dl[q] = t + (int32_t)budget;                  // PAPER.md:117 deadline = t_arrive + beta
                q_arr[q] = t;
                const uint32_t g = row_gid(P.plan, region, pidx0 + lane);
                P.plan.env[g] = e;
                P.plan.a[g] = q | (t_rel << 19);
                P.plan.b[g] = __fdiv_rn(__uint2float_rn(budget), __uint2float_rn(P.budget_norm));
                P.plan.c[g] = in_tok;
            }
            __syncwarp();
            if (lane < n_ok) atomicAnd(&S.qfree[q >> 5], ~(1u << (q & 31)));
            __syncwarp();
            c_live_mid += (lane == 0) ? (QCAP - n_free + n_ok) : 0;
        }
    }
    // ---- B snapshot (R14): telemetry features of the state left by the tick just finished
    if (pre_mode != 0 && lane < N) {
        float *sn = P.snap + (size_t)e * 3 * N;
        sn[lane] = __uint2float_rn(s_nwait[lane]) * 0x1p-6f;
        sn[N + lane] = __uint2float_rn(s_ewma[lane]) * 0x1p-18f;
        sn[2 * N + lane] = __fmul_rn(__uint2float_rn(s_kv[lane]), s_model[lane].kv_inv);
    }

    // ---- write back the small state
    __syncwarp();
    for (uint32_t w = lane; w < RW; w += 32) P.r_free[(size_t)e * RW + w] = S.rfree_new[w];
    for (uint32_t w = lane; w < QW; w += 32) { P.q_free[(size_t)e * QW + w] = S.qfree[w]; P.q_ready[(size_t)e * QW + w] = S.qready[w]; }
    if (lane < N) P.m_cnt[(size_t)e * N + lane] = make_uint4(s_nwait[lane], s_nrun[lane], s_kv[lane], s_ewma[lane]);
    if (lane == 0 && pre_mode == 1) P.e_hdr[e] = drops_next;
    {
        const uint32_t vals[16] = {c_arrivals, c_dropped, c_finished, c_solved, c_missed, c_issued, c_done, c_preempt,
                                   c_sojourn, c_live_mid, c_plans, c_issued, c_running, c_waiting, 0u, c_abandoned};
        uint32_t mine = 0;
#pragma unroll
        for (int i = 0; i < 16; i++) { const uint32_t s = warp_sum(vals[i]); if (lane == (uint32_t)i) mine = s; }
        if (lane < 16 && mine) P.counters[(size_t)e * 16 + lane] += mine;
    }
}

void launch_sim(const Params &P, int32_t t_post, uint32_t trow_post, int32_t t_pre, uint32_t pre_mode, int32_t t0, cudaStream_t st)
{
    const size_t smem = kSimWarps * sim_warp_smem_bytes(P.RCAP, P.QCAP);
    static bool attr_set = false;
    if (!attr_set) { cudaFuncSetAttribute(k_sim, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024); attr_set = true; }
    const uint32_t blocks = (P.E + kSimWarps - 1) / kSimWarps;
    k_sim<<<blocks, kSimWarps * 32, smem, st>>>(P, t_post, trow_post, t_pre, pre_mode, t0);
}

}  // namespace im
