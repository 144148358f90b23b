// im_sim.cu — the fixed-tick simulation kernel: one group of G lanes (a warp or a half-warp) per environment.
//
// One launch runs, for every env, the environment half of the canonical tick:
//   post(t):  D-issue (requests of the decisions the executor kernel took for tick t), E admit (slack-ordered
//             queue, R20/R21), F serve (token-level service, R11), G complete (latency, cost, EWMA, finalise,
//             R13/R27/R28), H preempt (R21), I record (R27/R28/R33)
//   pre(t+1): A arrive (Poisson count, budgets, input tokens; R5-R9), B snapshot (R14), and the emission of the
//             work lists: one planner row per new query, executor rows for every query whose previous stage
//             completed (R17).
// The decision half (C plan, D decide) runs between two launches in im_policy.cu.
//
// Shape of the work: the only O(pool) work of a tick is ONE streaming pass over hot[0..hwm) —
// 128-bit coalesced loads, one Philox call per 4 slots — which serves every RUNNING request, buckets the WAITING
// requests of the models that can admit, and lists the requests that completed.  Everything else (issue, admission,
// completion, preemption, arrivals) touches only the few requests that change state, in batches across the lanes so
// that a phase costs one memory round trip, not one per request.  Order-dependent definitions (j-th new item takes the
// j-th lowest free index, R9/R18; smallest key first, R20) are computed by ranked selection / repeated arg-min, every
// accumulation is an integer sum, so lanes may commit in any order (R12, R13, R28).
#include "im_device.cuh"

namespace im {

constexpr int kSimThreads = 128;

// ---- per-group shared memory layout (bytes)
struct SimLayout {
    uint32_t o_hdr, o_prefA, o_prefB, o_small, o_bucket, o_clist, total;
};
constexpr uint32_t kSmallWords = 9 * 16 + 8;
__host__ __device__ inline SimLayout sim_layout(uint32_t hdr_words, uint32_t RW, uint32_t QW, uint32_t RCAP, uint32_t G)
{
    auto up = [](uint32_t x) { return (x + 15u) & ~15u; };
    SimLayout L;
    uint32_t o = 0;
    L.o_hdr = o; o += up(hdr_words * 4);
    L.o_prefA = o; o += up((RW + 1) * 4);
    L.o_prefB = o; o += up((QW + 1) * 4);
    L.o_small = o; o += up(kSmallWords * 4);
    L.o_bucket = o; o += up(RCAP * 2);
    L.o_clist = o; o += up(5 * G * 2);
    L.total = o;
    return L;
}

template <int G>
struct Grp {
    uint32_t gl, gmask, gbase, lane;
    __device__ __forceinline__ uint32_t ballot(bool p) const
    {
        const uint32_t b = __ballot_sync(gmask, p) >> gbase;
        return G == 32 ? b : (b & ((1u << (G & 31)) - 1u));
    }
    template <typename T> __device__ __forceinline__ T shfl(T v, int src) const { return __shfl_sync(gmask, v, src, G); }
    template <typename T> __device__ __forceinline__ T shfl_up(T v, int d) const { return __shfl_up_sync(gmask, v, d, G); }
    template <typename T> __device__ __forceinline__ T shfl_xor(T v, int d) const { return __shfl_xor_sync(gmask, v, d, G); }
    __device__ __forceinline__ void sync() const { __syncwarp(gmask); }
    __device__ __forceinline__ uint32_t incl_scan(uint32_t v) const
    {
#pragma unroll
        for (int o = 1; o < G; o <<= 1) { const uint32_t n = shfl_up(v, o); if (gl >= (uint32_t)o) v += n; }
        return v;
    }
    __device__ __forceinline__ uint32_t sum(uint32_t v) const { return __reduce_add_sync(gmask, v); }
    __device__ __forceinline__ uint32_t umin(uint32_t v) const { return __reduce_min_sync(gmask, v); }
    __device__ __forceinline__ uint32_t umax(uint32_t v) const { return __reduce_max_sync(gmask, v); }
};

// exclusive prefix of popcounts of bm[0..nw) into pref[0..nw]; returns the total
template <int G>
__device__ __forceinline__ uint32_t build_prefix(const Grp<G> &g, const uint32_t *bm, uint32_t nw, uint32_t *pref)
{
    uint32_t carry = 0;
    for (uint32_t w0 = 0; w0 < nw; w0 += G) {
        const uint32_t w = w0 + g.gl;
        const uint32_t pc = w < nw ? __popc(bm[w]) : 0u;
        const uint32_t inc = g.incl_scan(pc);
        if (w < nw) pref[w] = carry + inc - pc;
        carry += g.shfl(inc, G - 1);
    }
    if (g.gl == 0) pref[nw] = carry;
    g.sync();
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

// tick arguments: t_post < 0 => no post phases; pre_mode 0 none, 1 full (A, B, rows), 2 snapshot only
template <int G>
__global__ void __launch_bounds__(kSimThreads)
k_sim(const Params P, int32_t t_post, uint32_t trow_post, int32_t t_pre, uint32_t pre_mode, int32_t t0)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ ModelTab s_model[kMaxModels];
    __shared__ uint32_t s_base[kMaxModels], s_frac[kMaxModels];
    if (threadIdx.x < P.N) {
        s_model[threadIdx.x] = P.model[threadIdx.x];
        const uint32_t x = P.model[threadIdx.x].rate * kDtUs;            // rate <= 80000 => fits 32 bits
        s_base[threadIdx.x] = x / 1000000u; s_frac[threadIdx.x] = x % 1000000u;
    }
    __syncthreads();
    constexpr uint32_t GPB = kSimThreads / G;
    Grp<G> g;
    g.lane = threadIdx.x & 31; g.gl = threadIdx.x % G; g.gbase = g.lane - g.gl;
    g.gmask = G == 32 ? 0xffffffffu : (((1u << (G & 31)) - 1u) << g.gbase);
    const uint32_t gl = g.gl;
    const uint32_t e = blockIdx.x * GPB + threadIdx.x / G;
    if (e >= P.E) return;
    const uint32_t gid = P.env_id_base + e;
    const uint32_t N = P.N, RW = P.RW, QW = P.QW, RCAP = P.RCAP, QCAP = P.QCAP;
    const uint32_t region = e % kRegions;

    const SimLayout L = sim_layout(P.hdr_words, RW, QW, RCAP, G);
    unsigned char *sm = smem_raw + (size_t)(threadIdx.x / G) * L.total;
    uint32_t *s_hdr = (uint32_t *)(sm + L.o_hdr);
    uint32_t *s_rfree = s_hdr + P.hw_rfree, *s_qfree = s_hdr + P.hw_qfree, *s_qready = s_hdr + P.hw_qready, *s_misc = s_hdr + P.hw_misc;
    uint32_t *prefA = (uint32_t *)(sm + L.o_prefA), *prefB = (uint32_t *)(sm + L.o_prefB);
    uint32_t *s_small = (uint32_t *)(sm + L.o_small);
    uint32_t *s_boff = s_small, *s_bcnt = s_small + 16, *s_latsum = s_small + 32, *s_latn = s_small + 48;
    int32_t *s_kvcorr = (int32_t *)(s_small + 64);
    uint32_t *s_relkv = s_small + 80, *s_relnrun = s_small + 96, *s_ext = s_small + 112, *s_ctr = s_small + 128;
    uint32_t *s_sc = s_small + 144;                  // [0] ccnt, [1] rew, [2] miss, [4..5] cost (u64)
    unsigned long long *s_cost = (unsigned long long *)(s_sc + 4);
    uint16_t *s_bucket = (uint16_t *)(sm + L.o_bucket), *s_clist = (uint16_t *)(sm + L.o_clist);

    uint8_t *rec = env_rec(P, e);
    uint32_t *hot = (uint32_t *)(rec + P.off_hot), *r_tok = (uint32_t *)(rec + P.off_tok), *r_aux = (uint32_t *)(rec + P.off_aux);
    int32_t *r_dl = (int32_t *)(rec + P.off_dl), *r_issue = (int32_t *)(rec + P.off_issue);
    uint4 *qtab = (uint4 *)(rec + P.off_q);

    // ---- load the header
    {
        const uint4 *src = (const uint4 *)rec;
        uint4 *dst = (uint4 *)s_hdr;
        for (uint32_t i = gl; i < P.hdr_words / 4; i += G) dst[i] = src[i];
        for (uint32_t i = gl; i < kSmallWords; i += G) s_small[i] = 0;
    }
    g.sync();
#define M_NWAIT(k) s_hdr[4 * (k) + 0]
#define M_NRUN(k) s_hdr[4 * (k) + 1]
#define M_KV(k) s_hdr[4 * (k) + 2]
#define M_EWMA(k) s_hdr[4 * (k) + 3]

    // Emission of the executor rows of queries whose previous stage completed (R17): lanes with `valid` hold one query.
    auto emit_ready = [&](bool valid, uint32_t q, uint32_t pw, uint32_t in_tok, int32_t dl, uint32_t t_rel) {
        uint32_t a0 = 0, nc = 0;
        if (valid) stage_calls((pw >> 2) & 3u, (pw >> 6) & 7u, (pw >> 9) & 7u, a0, nc);
        const uint32_t inc = g.incl_scan(nc);
        const uint32_t tot = g.shfl(inc, G - 1);
        if (tot == 0) return;
        uint32_t idx0 = 0;
        if (gl == 0) idx0 = rows_claim(P, P.exec, region, tot);
        idx0 = g.shfl(idx0, 0) + inc - nc;
        if (valid) {
            write_exec_rows(P, region, idx0, e, q, pw, in_tok, dl, t_rel, a0, nc);
            // stage++, pending = nc: the calls are issued in phase D of the coming tick
            qtab[q].x = (pw & ~((7u << 9) | (3u << QP_PEND_SHIFT))) | ((((pw >> 9) & 7u) + 1u) << 9) | (nc << QP_PEND_SHIFT);
        }
    };

    if (t_post >= 0) {
        const int32_t t = t_post;
        const uint32_t done = (P.episode_ticks && ((uint32_t)(t + 1) % P.episode_ticks) == 0) ? 1u : 0u;
        const bool emit = (pre_mode == 1) && !done;
        const uint32_t t_rel_next = (uint32_t)(t + 1 - t0);

        // ---- G complete for a batch of <= G listed requests (R1, R13, R27, R28)
        auto flush = [&]() {
            const uint32_t ccnt = s_sc[0];
            const uint32_t nb = ccnt < (uint32_t)G ? ccnt : (uint32_t)G;
            const bool act = gl < nb;
            uint32_t q = 0x10000u + gl, model = 0, succ = 0;
            uint4 qr = make_uint4(0, 0, 0, 0);
            if (act) {
                const uint32_t ent = s_clist[ccnt - nb + gl];
                const uint32_t ridx = ent & 0xFFFu;
                model = ent >> 12;
                const int32_t issue = r_issue[ridx];
                const uint32_t tk = r_tok[ridx], aux = r_aux[ridx];
                q = aux >> 16; succ = (aux >> 10) & 1u;
                qr = qtab[q];
                const uint32_t ell = (uint32_t)(t + 1 - issue);
                atomicAdd(s_cost, ((unsigned long long)ell << 16) / (qr.y & 0xFFFFu));   // C_k = l_k / beta, Q16 (R28)
                atomicAdd(&s_latsum[model], ell); atomicAdd(&s_latn[model], 1u);
                atomicAdd(&s_relkv[model], (tk >> 16) + (tk & 0xFFFFu)); atomicAdd(&s_relnrun[model], 1u);
                atomicAdd(&s_ctr[C_CALLS_DONE], 1u);
            }
            // calls of one query that complete in the same tick are folded by the lowest lane holding them
            const uint32_t peers = __match_any_sync(g.gmask, q);
            const uint32_t succm = __ballot_sync(g.gmask, act && succ);
            const bool leader = act && ((uint32_t)(__ffs(peers) - 1) == g.lane);
            bool fin = false, ready = false;
            uint32_t pw = qr.x;
            if (leader) {
                const uint32_t pend = ((pw >> QP_PEND_SHIFT) & 3u) - (uint32_t)__popc(peers);
                pw = (pw & ~(3u << QP_PEND_SHIFT)) | (pend << QP_PEND_SHIFT) | (((succm & peers) ? 1u : 0u) << QP_SUCC_SHIFT);
                if (pend == 0) { if (((pw >> 9) & 7u) == ((pw >> 12) & 7u)) fin = true; else ready = true; }
                if (!fin && !(ready && emit)) qtab[q].x = pw;
                if (ready && !emit) atomicOr(&s_qready[q >> 5], 1u << (q & 31));
            }
            // finalise (R27): reward, SLO miss, sojourn, query log
            const uint32_t finm = g.ballot(fin);
            if (finm) {
                uint32_t lbase = 0;
                if (gl == 0) {
                    lbase = atomicAdd(&P.qlog.cnt[region], (uint32_t)__popc(finm));
                    if (lbase + __popc(finm) > P.qlog.regcap) atomicOr(P.err_flag, 2u);
                }
                lbase = g.shfl(lbase, 0);
                if (fin) {
                    const uint32_t solved = (pw >> QP_SUCC_SHIFT) & 1u;
                    const uint32_t sojourn = (uint32_t)(t + 1 - (int32_t)qr.w);
                    const uint32_t late = (t + 1 > (int32_t)qr.z) ? 1u : 0u;
                    atomicAdd(&s_sc[1], solved); atomicAdd(&s_sc[2], late);
                    atomicAdd(&s_ctr[C_FINISHED], 1u); atomicAdd(&s_ctr[C_SOLVED], solved); atomicAdd(&s_ctr[C_MISSED], late);
                    atomicAdd(&s_ctr[C_SUM_SOJOURN], sojourn);
                    const uint32_t li = lbase + __popc(finm & ((1u << gl) - 1u));
                    P.qlog.rec[(size_t)region * P.qlog.regcap + (li % P.qlog.regcap)] =
                        make_uint4(gid, qr.w, sojourn, (qr.y & 0xFFFFu) | (solved << 16) | (((pw >> 2) & 3u) << 17) | (((pw >> 6) & 7u) << 19));
                    atomicOr(&s_qfree[q >> 5], 1u << (q & 31));
                }
            }
            if (emit && g.ballot(ready)) emit_ready(ready, q, pw, qr.y >> 16, (int32_t)qr.z, t_rel_next);
            g.sync();
            if (gl == 0) s_sc[0] = ccnt - nb;
            g.sync();
        };

        // =============================================================== D-issue (R18): canonical request indices
        const uint32_t icnt = min(s_misc[1], kIssueCap);        // the executor kernel flags an overflow (err_flag)
        if (icnt) {
            const uint4 *iss = (const uint4 *)(rec + P.off_iss);
            build_prefix(g, s_rfree, RW, prefA);
            uint16_t *skey = s_bucket;                        // scratch: (q << 2 | agent) of every record
            for (uint32_t j = gl; j < icnt; j += G) { const uint32_t aux = iss[j].y; skey[j] = (uint16_t)(((aux >> 16) << 2) | ((aux >> 8) & 3u)); }
            g.sync();
            for (uint32_t j = gl; j < icnt; j += G) {
                const uint4 r = iss[j];
                const uint32_t key = skey[j];
                uint32_t rank = 0;
                for (uint32_t i = 0; i < icnt; i++) rank += skey[i] < key ? 1u : 0u;
                const uint32_t ridx = find_nth(s_rfree, RW, prefA, rank);
                const uint32_t model = (r.y >> 2) & 15u;
                r_tok[ridx] = r.x; r_aux[ridx] = r.y; r_dl[ridx] = (int32_t)r.z; r_issue[ridx] = t;
                hot[ridx] = (r.x & 0xFFFFu) | (ST_WAIT << HOT_STATE_SHIFT) | (model << HOT_MODEL_SHIFT);
                atomicAdd(&M_NWAIT(model), 1u);
            }
            g.sync();
            // the icnt lowest free indices are exactly the ones taken: clear them word by word
            for (uint32_t w = gl; w < RW; w += G) {
                const uint32_t before = prefA[w], cntw = prefA[w + 1] - before;
                if (before < icnt) {
                    const uint32_t take = min(icnt - before, cntw);
                    uint32_t bm = s_rfree[w];
                    if (take == cntw) bm = 0; else for (uint32_t i = 0; i < take; i++) bm &= bm - 1;
                    s_rfree[w] = bm;
                }
            }
            if (gl == 0) { s_ctr[C_ISSUED] += icnt; s_ctr[C_EXEC_DEC] += icnt; s_misc[1] = 0; }
            g.sync();
        }
        // high-water mark of the request pool (highest occupied index + 1)
        uint32_t hwm = 0;
        for (uint32_t w = gl; w < RW; w += G) {
            const uint32_t occ = ~s_rfree[w];
            if (occ) hwm = max(hwm, w * 32 + 32 - __clz(occ));
        }
        hwm = g.umax(hwm);
        const uint32_t n_chunks = (hwm + 4 * G - 1) / (4 * G);

        // models that can admit (R21) and the offsets of their buckets
        const bool adm = gl < N && M_NWAIT(gl) > 0 && M_NRUN(gl) < s_model[gl].slots && M_KV(gl) <= s_model[gl].kv_cap;
        const uint32_t madm = g.ballot(adm);
        const uint32_t nrun_pre = gl < N ? M_NRUN(gl) : 0u;
        {
            const uint32_t nw = adm ? M_NWAIT(gl) : 0u;
            const uint32_t inc = g.incl_scan(nw);
            if (gl < 16) s_boff[gl] = inc - nw;
        }
        g.sync();

        // =============================================================== F serve (R11): one streaming pass over hot[0..hwm)
        unsigned long long ext_lo = 0, ext_hi = 0;             // per-lane count of stochastic extra tokens, 8 bits per model
        {
            uint4 *hot4 = (uint4 *)hot;
            uint4 hn = make_uint4(0, 0, 0, 0);
            if (n_chunks) hn = hot4[gl];
            for (uint32_t c = 0; c < n_chunks; c++) {
                const uint32_t i0 = (c * G + gl) * 4;
                const uint4 h4 = hn;
                if (c + 1 < n_chunks) hn = hot4[(c + 1) * G + gl];
                uint32_t hh[4] = {h4.x, h4.y, h4.z, h4.w};
                {   // free slots are defined by the bitmap: their words may be stale (reset, episode boundary)
                    const uint32_t fr = s_rfree[i0 >> 5] >> (i0 & 31);
#pragma unroll
                    for (int s = 0; s < 4; s++) if ((fr >> s) & 1u) hh[s] = 0;
                }
                const uint32_t stor = (hh[0] | hh[1] | hh[2] | hh[3]) >> HOT_STATE_SHIFT;   // any non-free slot?
                bool dirty = false;
                if (stor & 3u) {
                    const bool any_run = (((hh[0] >> 17) | (hh[1] >> 17) | (hh[2] >> 17) | (hh[3] >> 17)) & 1u) != 0;
                    Ph4 u4 = Ph4{0, 0, 0, 0};
                    if (any_run) u4 = draw(P, STREAM_SVC, gid, t, i0 >> 2, 0);
                    const uint32_t uu[4] = {u4.x, u4.y, u4.z, u4.w};
#pragma unroll
                    for (int s = 0; s < 4; s++) {
                        const uint32_t w = hh[s];
                        const uint32_t st = (w >> HOT_STATE_SHIFT) & 3u, model = (w >> HOT_MODEL_SHIFT) & 15u;
                        if (st == ST_RUN) {
                            const uint32_t rem = w & 0xFFFFu;
                            const uint32_t extra = __umulhi(uu[s], 1000000u) < s_frac[model] ? 1u : 0u;
                            const uint32_t tok = s_base[model] + extra;
                            if (model < 8) ext_lo += (unsigned long long)extra << (8 * model); else ext_hi += (unsigned long long)extra << (8 * (model - 8));
                            if (tok >= rem) {                                    // completes: only `rem` tokens are decoded
                                if (tok != rem) atomicAdd(&s_kvcorr[model], (int32_t)rem - (int32_t)tok);
                                const uint32_t pos = atomicAdd(&s_sc[0], 1u);
                                s_clist[pos] = (uint16_t)((model << 12) | (i0 + s));
                                atomicOr(&s_rfree[(i0 + s) >> 5], 1u << ((i0 + s) & 31));
                                hh[s] = 0;
                            } else {
                                hh[s] = w - tok;
                            }
                            dirty = true;
                        } else if (st == ST_WAIT && ((madm >> model) & 1u)) {
                            const uint32_t pos = s_boff[model] + atomicAdd(&s_bcnt[model], 1u);
                            s_bucket[pos] = (uint16_t)((model << 12) | (i0 + s));
                        }
                    }
                }
                if (dirty) hot4[c * G + gl] = make_uint4(hh[0], hh[1], hh[2], hh[3]);
                g.sync();
                while (s_sc[0] >= (uint32_t)G) flush();
            }
        }
        // per-model totals of the extra tokens
        {
            const uint32_t lo0 = (uint32_t)ext_lo, lo1 = (uint32_t)(ext_lo >> 32), hi0 = (uint32_t)ext_hi, hi1 = (uint32_t)(ext_hi >> 32);
            const uint32_t v[8] = {lo0 & 0x00FF00FFu, (lo0 >> 8) & 0x00FF00FFu, lo1 & 0x00FF00FFu, (lo1 >> 8) & 0x00FF00FFu,
                                   hi0 & 0x00FF00FFu, (hi0 >> 8) & 0x00FF00FFu, hi1 & 0x00FF00FFu, (hi1 >> 8) & 0x00FF00FFu};
            uint32_t r[8];
#pragma unroll
            for (int i = 0; i < 8; i++) r[i] = g.sum(v[i]);
            if (gl == 0) {
#pragma unroll
                for (int i = 0; i < 8; i++) {
                    const int m0 = (i >> 1) * 4 + (i & 1);       // v[i] holds models m0 (low half) and m0 + 2 (high half)
                    s_ext[m0] = r[i] & 0xFFFFu; s_ext[m0 + 2] = r[i] >> 16;
                }
            }
        }
        g.sync();

        // =============================================================== E admit (R20, R21): smallest key first, per model
        {
            uint32_t mleft = madm;
            while (mleft) {
                const uint32_t k = __ffs(mleft) - 1;
                mleft &= mleft - 1;
                const uint32_t off = s_boff[k], cnt = s_bcnt[k];
                uint32_t nw = M_NWAIT(k), nr = M_NRUN(k), kv = M_KV(k), tok_adm = 0;   // tokens served to this tick's admissions (phase F)
                const uint32_t slots = s_model[k].slots, cap = s_model[k].kv_cap;
                auto scan_min = [&](uint32_t last, bool first) {
                    uint32_t best = 0xFFFFFFFFu;
                    for (uint32_t j = gl; j < cnt; j += G) {
                        const uint32_t ridx = s_bucket[off + j] & 0xFFFu;
                        const int32_t bt = P.sched_mode ? r_dl[ridx] : r_issue[ridx];
                        const uint32_t key = ((uint32_t)(bt - t + (1 << 19)) << 12) | ridx;
                        if ((first || key > last) && key < best) best = key;
                    }
                    return best;
                };
                uint32_t best = scan_min(0, true);
                for (;;) {
                    const uint32_t wkey = g.umin(best);
                    if (wkey == 0xFFFFFFFFu) break;
                    const uint32_t ridx = wkey & 0xFFFu;
                    const uint32_t tk = r_tok[ridx], hw = hot[ridx];
                    uint32_t rem = hw & 0xFFFFu;
                    const uint32_t need = (tk >> 16) + ((tk & 0xFFFFu) - rem);           // R12
                    if (!(nr < slots && kv + need <= cap)) break;                         // stop at the first misfit (R21)
                    // admitted: prefill, then its first tick of service (R11)
                    const uint32_t pf = (uint32_t)(((unsigned long long)s_model[k].prefill * need) / 1000u);
                    const uint32_t usable = kDtUs - min(pf, kDtUs);
                    const uint32_t x = s_model[k].rate * usable;
                    const uint32_t bs = x / 1000000u, fr = x - bs * 1000000u;
                    const Ph4 u4 = draw(P, STREAM_SVC, gid, t, ridx >> 2, 0);
                    const uint32_t uu = (ridx & 3u) == 0 ? u4.x : ((ridx & 3u) == 1 ? u4.y : ((ridx & 3u) == 2 ? u4.z : u4.w));
                    const uint32_t tok = min(bs + (__umulhi(uu, 1000000u) < fr ? 1u : 0u), rem);
                    rem -= tok;
                    kv += need; tok_adm += tok; nw -= 1; nr += 1;
                    if (gl == 0) {
                        if (rem == 0) {
                            s_clist[s_sc[0]] = (uint16_t)((k << 12) | ridx);
                            s_sc[0] += 1;
                            s_rfree[ridx >> 5] |= 1u << (ridx & 31);
                            hot[ridx] = 0;
                        } else {
                            hot[ridx] = rem | (ST_RUN << HOT_STATE_SHIFT) | (k << HOT_MODEL_SHIFT);
                        }
                    }
                    if (rem == 0) {
                        g.sync();
                        while (s_sc[0] >= (uint32_t)G) flush();
                    }
                    if (nw == 0 || nr >= slots) break;
                    if (best == wkey) best = scan_min(wkey, false);
                }
                if (gl == 0) { M_NWAIT(k) = nw; M_NRUN(k) = nr; M_KV(k) = kv + tok_adm; }
            }
            g.sync();
        }
        // service totals of the requests that were RUNNING before this tick's admissions
        if (gl < N) M_KV(gl) = (uint32_t)((int32_t)(M_KV(gl) + nrun_pre * s_base[gl] + s_ext[gl]) + s_kvcorr[gl]);
        g.sync();

        // =============================================================== G complete: the rest of the list, then EWMA (R13)
        while (s_sc[0] > 0) flush();
        if (gl < N) {
            M_KV(gl) -= s_relkv[gl]; M_NRUN(gl) -= s_relnrun[gl];
            if (s_latn[gl] > 0) {
                const int32_t mean_q8 = (int32_t)((s_latsum[gl] << 8) / s_latn[gl]);
                int32_t ew = (int32_t)M_EWMA(gl);
                ew += (mean_q8 - ew) >> 3;
                M_EWMA(gl) = (uint32_t)ew;
            }
        }
        g.sync();

        // =============================================================== H preempt (R21)
        if (P.kv_preempt) {
            uint32_t mover = g.ballot(gl < N && M_KV(gl) > s_model[gl].kv_cap);
            while (mover) {
                const uint32_t k = __ffs(mover) - 1;
                mover &= mover - 1;
                // list the RUNNING requests of model k (second pass over hot, now in L2)
                if (gl == 0) s_bcnt[0] = 0;
                g.sync();
                const uint4 *hot4 = (const uint4 *)hot;
                for (uint32_t c = 0; c < n_chunks; c++) {
                    const uint32_t i0 = (c * G + gl) * 4;
                    const uint4 h4 = hot4[c * G + gl];
                    const uint32_t hh[4] = {h4.x, h4.y, h4.z, h4.w};
                    const uint32_t fr = s_rfree[i0 >> 5] >> (i0 & 31);
#pragma unroll
                    for (int s = 0; s < 4; s++)
                        if (!((fr >> s) & 1u) && ((hh[s] >> HOT_STATE_SHIFT) & 3u) == ST_RUN && ((hh[s] >> HOT_MODEL_SHIFT) & 15u) == k)
                            s_bucket[atomicAdd(&s_bcnt[0], 1u)] = (uint16_t)(i0 + s);
                }
                g.sync();
                const uint32_t cnt = s_bcnt[0];
                uint32_t kv = M_KV(k), nr = M_NRUN(k), nw = M_NWAIT(k), npre = 0;
                // victim = largest (deadline, ridx); candidates strictly below the previous victim on later rounds
                auto scan_max = [&](uint32_t lim_d, uint32_t lim_i, bool first, uint32_t &bd, uint32_t &bi) {
                    bd = 0; bi = 0; bool have = false;
                    for (uint32_t j = gl; j < cnt; j += G) {
                        const uint32_t ridx = s_bucket[j];
                        const uint32_t d = (uint32_t)r_dl[ridx] + 0x80000000u;
                        const bool below = first || d < lim_d || (d == lim_d && ridx < lim_i);
                        if (below && (!have || d > bd || (d == bd && ridx > bi))) { bd = d; bi = ridx; have = true; }
                    }
                    return have;
                };
                uint32_t bd, bi;
                bool have = scan_max(0, 0, true, bd, bi);
                while (kv > s_model[k].kv_cap) {
                    if (!g.ballot(have)) break;
                    const uint32_t wd = g.umax(have ? bd : 0u);
                    const uint32_t wi = g.umax((have && bd == wd) ? bi + 1u : 0u) - 1u;
                    const uint32_t tk = r_tok[wi], hw = hot[wi];
                    kv -= (tk >> 16) + ((tk & 0xFFFFu) - (hw & 0xFFFFu));
                    nr -= 1; nw += 1; npre += 1;
                    if (gl == 0) hot[wi] = (hw & ~(3u << HOT_STATE_SHIFT)) | (ST_WAIT << HOT_STATE_SHIFT);
                    if (have && bd == wd && bi == wi) have = scan_max(wd, wi, false, bd, bi);
                }
                if (gl == 0) { M_KV(k) = kv; M_NRUN(k) = nr; M_NWAIT(k) = nw; s_ctr[C_PREEMPT] += npre; }
                g.sync();
            }
        }

        // =============================================================== I record (R27, R28, R33)
        {
            const uint32_t drops = s_misc[0];                   // R9: drops of this tick's phase A
            const uint32_t miss_acc = s_sc[2] + drops;
            const unsigned long long cost_acc = *s_cost + ((unsigned long long)drops << 16);
            if (gl == 0) {
                const size_t idx = (size_t)trow_post * P.E + e;
                P.rew[idx] = __uint2float_rn(s_sc[1]);
                P.cost[idx] = P.cost_mode ? __uint2float_rn(miss_acc) : __ull2float_rn(cost_acc) * 0x1p-16f;
                P.miss[idx] = (uint8_t)min(miss_acc, 255u);
                P.done[idx] = (uint8_t)done;
            }
            const uint32_t nr_sum = g.sum(gl < N ? M_NRUN(gl) : 0u), nw_sum = g.sum(gl < N ? M_NWAIT(gl) : 0u);
            if (gl == 0) { s_ctr[C_SUM_RUNNING] += nr_sum; s_ctr[C_SUM_WAITING] += nw_sum; }
            g.sync();
            if (done) {
                // hard reset: live queries abandoned, tables emptied (free slots are defined by the bitmaps)
                uint32_t live = 0;
                for (uint32_t w = gl; w < QW; w += G) live += __popc(~s_qfree[w]);
                live = g.sum(live);
                if (gl == 0) s_ctr[C_ABANDONED] += live;
                for (uint32_t w = gl; w < RW; w += G) s_rfree[w] = 0xFFFFFFFFu;
                for (uint32_t w = gl; w < QW; w += G) { s_qfree[w] = 0xFFFFFFFFu; s_qready[w] = 0; }
                if (gl < N) { M_NWAIT(gl) = 0; M_NRUN(gl) = 0; M_KV(gl) = 0; M_EWMA(gl) = 0; }
            }
            if (gl == 0) s_misc[0] = 0;
            g.sync();
        }
    }

    // ===================================================================== pre(t_pre): A arrive, B snapshot, work lists
    if (pre_mode == 1) {
        const int32_t t = t_pre;
        const uint32_t t_rel = (uint32_t)(t - t0);
        // ---- executor rows of queries left ready by an earlier rollout (pending == 0, stages left)
        {
            const uint32_t n_ready = build_prefix(g, s_qready, QW, prefB);
            for (uint32_t b0 = 0; b0 < n_ready; b0 += G) {
                const uint32_t o = b0 + gl;
                uint32_t q = 0;
                uint4 qr = make_uint4(0, 0, 0, 0);
                if (o < n_ready) { q = find_nth(s_qready, QW, prefB, o); qr = qtab[q]; }
                emit_ready(o < n_ready, q, qr.x, qr.y >> 16, (int32_t)qr.z, t_rel);
            }
            g.sync();
            if (n_ready) for (uint32_t w = gl; w < QW; w += G) s_qready[w] = 0;
            g.sync();
        }
        // ---- A arrive (R5, R7, R8, R9)
        {
            const uint32_t xr = draw(P, STREAM_ARR, gid, t, 0, 0).x;
            const uint32_t *cdf = P.tab_cdf + 32u * P.env_level[e];
            uint32_t n = 0;
            for (uint32_t j = gl; j < 31; j += G) n += xr >= __ldg(&cdf[j]) ? 1u : 0u;
            n = g.sum(n);
            const uint32_t n_free = build_prefix(g, s_qfree, QW, prefB);
            const uint32_t n_ok = min(n, n_free);
            uint32_t pidx0 = 0;
            if (gl == 0 && n_ok) pidx0 = rows_claim(P, P.plan, region, n_ok);
            pidx0 = g.shfl(pidx0, 0);
            for (uint32_t j = gl; j < n_ok; j += G) {
                const uint32_t q = find_nth(s_qfree, QW, prefB, j);
                const Ph4 d = draw(P, STREAM_QRY, gid, t, j, 0);
                const uint32_t comp = d.z < P.mix_thresh ? 0u : 1u;
                const uint32_t budget = P.mix_lo[comp] + __umulhi(d.x, P.mix_hi[comp] - P.mix_lo[comp] + 1u);
                const uint32_t in_tok = P.has_intok ? __ldg(&P.tab_intok[d.y >> 22]) : P.in_tok_const;
                const int32_t dl = t + (int32_t)budget;                  // PAPER.md:117 deadline = t_arrive + beta
                qtab[q] = make_uint4(QP_LIVE, budget | (in_tok << 16), (uint32_t)dl, (uint32_t)t);
                P.plan.row[row_gid(P.plan, region, pidx0 + j)] = make_uint4(e, q | (t_rel << 19), (uint32_t)dl, in_tok);
            }
            g.sync();
            // the n_ok lowest free query indices are the ones taken
            for (uint32_t w = gl; w < QW; w += G) {
                const uint32_t before = prefB[w], cntw = prefB[w + 1] - before;
                if (before < n_ok) {
                    const uint32_t take = min(n_ok - before, cntw);
                    uint32_t bm = s_qfree[w];
                    if (take == cntw) bm = 0; else for (uint32_t i = 0; i < take; i++) bm &= bm - 1;
                    s_qfree[w] = bm;
                }
            }
            if (gl == 0) {
                s_ctr[C_ARRIVALS] += n; s_ctr[C_DROPPED] += n - n_ok; s_ctr[C_PLANS] += n_ok;
                s_ctr[C_SUM_LIVE_MID] += QCAP - n_free + n_ok;
                s_misc[0] = n - n_ok;                                   // drops carried to phase I of this tick
            }
            g.sync();
        }
    }
    // ---- B snapshot (R14): telemetry features of the state left by the tick just finished
    if (pre_mode != 0 && gl < N) {
        float *sn = P.snap + (size_t)e * 3 * N;
        sn[gl] = __uint2float_rn(M_NWAIT(gl)) * 0x1p-6f;
        sn[N + gl] = __uint2float_rn(M_EWMA(gl)) * 0x1p-18f;
        sn[2 * N + gl] = __fmul_rn(__uint2float_rn(M_KV(gl)), s_model[gl].kv_inv);
    }
    // ---- counters, then write the header back
    if (gl < 16 && s_ctr[gl]) {
        unsigned long long *c64 = (unsigned long long *)(s_hdr + P.hw_ctr);
        c64[gl] += s_ctr[gl];
    }
    g.sync();
    {
        uint4 *dst = (uint4 *)rec;
        const uint4 *src = (const uint4 *)s_hdr;
        for (uint32_t i = gl; i < P.hdr_words / 4; i += G) dst[i] = src[i];
    }
#undef M_NWAIT
#undef M_NRUN
#undef M_KV
#undef M_EWMA
}

void launch_sim(const Params &P, int32_t t_post, uint32_t trow_post, int32_t t_pre, uint32_t pre_mode, int32_t t0, cudaStream_t st)
{
    // a half-warp per env doubles the envs in flight at the same register footprint; the packed 8-bit extra-token
    // counters bound the slots one lane may serve to 255 (4 * RCAP / (4 * G) <= 255)
    const bool half = P.N <= 16 && P.RCAP / 16 <= 255;
    const uint32_t G = half ? 16 : 32;
    const SimLayout L = sim_layout(P.hdr_words, P.RW, P.QW, P.RCAP, G);
    const uint32_t gpb = kSimThreads / G;
    const size_t smem = (size_t)gpb * L.total;
    const uint32_t blocks = (P.E + gpb - 1) / gpb;
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(k_sim<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        cudaFuncSetAttribute(k_sim<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        attr_set = true;
    }
    if (half) k_sim<16><<<blocks, kSimThreads, smem, st>>>(P, t_post, trow_post, t_pre, pre_mode, t0);
    else k_sim<32><<<blocks, kSimThreads, smem, st>>>(P, t_post, trow_post, t_pre, pre_mode, t0);
}

}  // namespace im
