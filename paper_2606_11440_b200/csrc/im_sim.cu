// im_sim.cu — the fixed-tick simulation kernel: one group of G lanes (a half-warp) per environment, 24 envs per CTA.
//
// One launch runs, for every env, the environment half of the canonical tick:
//   post(t):  D-issue (the calls the executor kernel decided for tick t join the waiting list), E admit
//             (slack-ordered queue, R20/R21), F serve (token-level service, R11), G complete (latency, cost, EWMA,
//             finalise, R13/R27/R28), H preempt (R21), I record (R27/R28/R33)
//   pre(t+1): A arrive (Poisson count, budgets, input tokens; R5-R9), B snapshot (R14), and the emission of the
//             work lists: one planner row per new query, executor rows for every query whose previous stage
//             completed (R17).
// The decision half (C plan, D decide) runs between two launches in im_policy.cu.
//
// Shape of the work: the only O(pool) work of a tick is ONE streaming pass over hot[0..SP), the
// per-model service slots (R10) — 128-bit coalesced loads, a lane owns 8 consecutive slots of ONE model, one Philox
// call per 8 slots (sixteen-bit fields, R2/R11), no per-slot decode.  Everything else (issue, admission, completion,
// preemption, arrivals) touches only the few requests that change state.  The waiting list is a compact unordered
// array of u32 keys model|time|id: admission takes per-model minima of it (all admitting models in parallel, one lane
// per model), removal fills the holes from the tail.  Every accumulation is an integer sum, so lanes may commit in any
// order (R12, R13, R28).
#include "im_device.cuh"
#include <cstdlib>

namespace im {

constexpr int kSimThreads = 384;   // 3 CTAs per SM; measured on configs[4], ms per tick: (192,6) 0.714, (256,4) 0.686,
                                   // (320,4) 0.756, (352,3) 0.669, (384,3) 0.650, (416,3) 0.690, (448,2) 0.751

// ---- per-group shared memory layout (bytes)
struct SimLayout {
    uint32_t o_hdr, o_pref, o_small, o_clist, o_glist, total;
};
// small per-env arrays (u32 words): 16 per model-indexed array
enum : uint32_t { SM_LATSUM = 0, SM_LATN = 16, SM_RELKV = 32, SM_RELNRUN = 48, SM_KVADD = 64, SM_OCCCLR = 80, SM_AMIN = 112,
                  SM_AIDX = 128, SM_ALAST = 144, SM_CTR = 160, SM_SC = 176, SM_RM = 184, SM_MV = 200, kSmallWords = 216 };
inline SimLayout sim_layout(uint32_t hdr_words, uint32_t QW, uint32_t SP)
{
    auto up = [](uint32_t x) { return (x + 15u) & ~15u; };
    SimLayout L;
    uint32_t o = 0;
    L.o_hdr = o; o += up(hdr_words * 4);
    L.o_pref = o; o += up((QW + 1) * 4);
    L.o_small = o; o += up(kSmallWords * 4);
    L.o_clist = o; o += up(SP * 2);              // every slot may complete in one tick
    L.o_glist = o; o += 256;                     // non-empty slot groups of the tick: group | occupancy byte << 8
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
    __device__ __forceinline__ void sync() const { __syncwarp(gmask); }
    __device__ __forceinline__ uint32_t incl_scan(uint32_t v) const
    {
#pragma unroll
        for (int o = 1; o < G; o <<= 1) { const uint32_t n = shfl_up(v, o); if (gl >= (uint32_t)o) v += n; }
        return v;
    }
    __device__ __forceinline__ uint32_t sum(uint32_t v) const { return __reduce_add_sync(gmask, v); }
    __device__ __forceinline__ uint32_t umax(uint32_t v) const { return __reduce_max_sync(gmask, v); }
    __device__ __forceinline__ uint32_t umin(uint32_t v) const { return __reduce_min_sync(gmask, v); }
};

// exclusive prefix of popcounts of bm[0..nw) into pref[0..nw]; returns the total
template <int G>
__device__ __forceinline__ uint32_t build_prefix(const Grp<G> &g, const uint32_t *bm, uint32_t nw, uint32_t *pref)
{
    uint32_t carry = 0;
#pragma unroll 1
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
#pragma unroll 1
    while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (pref[mid] <= j) lo = mid; else hi = mid;
    }
    return lo * 32 + __fns(bm[lo], 0, (int)(j - pref[lo]) + 1);
}

// sixteen-bit field f (0..7) of a Philox output (R2: word f>>1, low half first)
__device__ __forceinline__ uint32_t u16_field(const Ph4 &u, uint32_t f)
{
    const uint32_t w = (f >> 1) == 0 ? u.x : ((f >> 1) == 1 ? u.y : ((f >> 1) == 2 ? u.z : u.w));
    return (f & 1u) ? (w >> 16) : (w & 0xFFFFu);
}

// tick arguments: t_post < 0 => no post phases; pre_mode 0 none, 1 full (A, B, rows), 2 snapshot only
template <int G>
__global__ void __launch_bounds__(kSimThreads, 3)
k_sim(const Params P, const SimLayout L, int32_t t_post, uint32_t trow_post, int32_t t_pre, uint32_t pre_mode, int32_t t0)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ ModelTab s_model[kMaxModels];
    __shared__ uint32_t s_base[kMaxModels], s_thr[kMaxModels], s_sbase[kMaxModels + 1];
    __shared__ uint8_t s_gmodel[128];                                       // group of 8 slots -> model
    if (threadIdx.x < P.N) {
        s_model[threadIdx.x] = P.model[threadIdx.x];
        const uint32_t x = P.model[threadIdx.x].rate * kDtUs;               // rate <= 80000 => fits 32 bits
        s_base[threadIdx.x] = x / 1000000u;
        s_thr[threadIdx.x] = (uint32_t)(((unsigned long long)(x % 1000000u) << 16) / 1000000u);   // R11: Bernoulli to 2^-16
    }
    if (threadIdx.x <= kMaxModels) s_sbase[threadIdx.x] = P.slot_base[threadIdx.x];
    if (threadIdx.x < (P.SP >> 3)) {
        uint32_t k = 0;
        while (P.slot_base[k + 1] <= threadIdx.x * 8) k++;
        s_gmodel[threadIdx.x] = (uint8_t)k;
    }
    __syncthreads();
    constexpr uint32_t GPB = kSimThreads / G;
    Grp<G> g;
    g.lane = threadIdx.x & 31; g.gl = threadIdx.x % G; g.gbase = g.lane - g.gl;
    g.gmask = G == 32 ? 0xffffffffu : (((1u << (G & 31)) - 1u) << g.gbase);
    const uint32_t gl = g.gl;
    const uint32_t lt_mask = (1u << gl) - 1u;
    // env blocks in descending order: neutral in general; where load rises with the env index (the utilisation sweep
    // of configs[3]-[4]) the heaviest CTAs start first and the last wave is the lightest (0.650 -> 0.643 ms per tick;
    // a level-interleaved order loses locality: 0.671)
    const uint32_t bid = gridDim.x - 1u - blockIdx.x;
    const uint32_t e = bid * GPB + threadIdx.x / G;
    if (e >= P.E) return;
    // The kernel is ~58 KB of code against a 32 KB instruction cache, and every group walks through all of it once per
    // tick.  Before the record / arrival phases (control flow there does not depend on the env) the groups of a CTA
    // wait for each other, so that the CTA's warps fetch the same lines at the same time (measured on configs[4] with
    // 384-thread CTAs, ms per tick: no barrier 0.721, before the service pass only 0.728, before the record only
    // 0.639, both 0.643; a second barrier before admission, completion or preemption: 0.649 / 0.654 / 0.647).
    const uint32_t cmask = (G == 32 || (e ^ 1u) >= P.E) ? g.gmask : 0xffffffffu;
    const bool cta_full = (bid + 1) * GPB <= P.E;
#define IM_CONVERGE() do { if (cta_full) __syncthreads(); else __syncwarp(cmask); } while (0)
#define IM_WCONV() __syncwarp(cmask)
    const uint32_t gid = P.env_id_base + e;
    const uint32_t N = P.N, QW = P.QW, QCAP = P.QCAP;
    const uint32_t region = e % kRegions;

    unsigned char *sm = smem_raw + (size_t)(threadIdx.x / G) * L.total;
    uint32_t *s_hdr = (uint32_t *)(sm + L.o_hdr);
    uint32_t *s_occ = s_hdr + P.hw_occ, *s_qfree = s_hdr + P.hw_qfree, *s_qready = s_hdr + P.hw_qready, *s_misc = s_hdr + P.hw_misc;
    uint32_t *prefB = (uint32_t *)(sm + L.o_pref);
    uint32_t *s_small = (uint32_t *)(sm + L.o_small);
    uint32_t *s_latsum = s_small + SM_LATSUM, *s_latn = s_small + SM_LATN, *s_relkv = s_small + SM_RELKV, *s_relnrun = s_small + SM_RELNRUN;
    uint32_t *s_kvadd = s_small + SM_KVADD, *s_occclr = s_small + SM_OCCCLR, *s_amin = s_small + SM_AMIN, *s_aidx = s_small + SM_AIDX;
    uint32_t *s_alast = s_small + SM_ALAST, *s_ctr = s_small + SM_CTR, *s_rm = s_small + SM_RM, *s_mv = s_small + SM_MV;
    uint32_t *s_sc = s_small + SM_SC;                 // [0] ccnt, [1] rew, [2] miss, [3] removals, [4..5] cost (u64)
    unsigned long long *s_cost = (unsigned long long *)(s_sc + 4);
    uint16_t *s_clist = (uint16_t *)(sm + L.o_clist); // completed requests: global slot index
    uint16_t *s_glist = (uint16_t *)(sm + L.o_glist);

    uint8_t *rec = env_rec(P, e);
    uint32_t *hot = (uint32_t *)(rec + P.off_hot), *wkey = (uint32_t *)(rec + P.off_wkey);
    uint2 *cold = (uint2 *)(rec + P.off_cold), *waux = (uint2 *)(rec + P.off_waux);
    uint4 *qtab = (uint4 *)(rec + P.off_q);

    // ---- load the header; the first group of slots of every lane is fetched with it (one round trip, not two)
    uint4 pre_a = make_uint4(0, 0, 0, 0), pre_b = pre_a;
    {
        const uint4 *src = (const uint4 *)rec;
        uint4 *dst = (uint4 *)s_hdr;
        const uint32_t nh = P.hdr_words / 4;                      // <= 49 uint4
        uint4 h0, h1, h2, h3;
        if (gl < nh) h0 = src[gl];
        if (gl + G < nh) h1 = src[gl + G];
        if (gl + 2 * G < nh) h2 = src[gl + 2 * G];
        if (gl + 3 * G < nh) h3 = src[gl + 3 * G];
        if (t_post >= 0 && gl < (P.SP >> 3)) { pre_a = ((const uint4 *)hot)[2 * gl]; pre_b = ((const uint4 *)hot)[2 * gl + 1]; }
#pragma unroll 1
        for (uint32_t i = gl; i < kSmallWords / 4; i += G) ((uint4 *)s_small)[i] = make_uint4(0, 0, 0, 0);
        if (gl < nh) dst[gl] = h0;
        if (gl + G < nh) dst[gl + G] = h1;
        if (gl + 2 * G < nh) dst[gl + 2 * G] = h2;
        if (gl + 3 * G < nh) dst[gl + 3 * G] = h3;
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
        if (gl == 0) idx0 = rows_claim(P, P.exec, region, tot) % P.exec.regcap;
        idx0 = g.shfl(idx0, 0) + inc - nc;
        if (idx0 >= P.exec.regcap) idx0 -= P.exec.regcap;
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
            uint32_t q = 0x10000u + gl, succ = 0;
            uint4 qr = make_uint4(0, 0, 0, 0);
            if (act) {
                const uint32_t gs = s_clist[ccnt - nb + gl], model = s_gmodel[gs >> 3], sl = gs - s_sbase[model];
                const uint2 cd = cold[gs];
                q = hot[gs] >> 18;                                           // id = 4 q + agent (the word was just written: L1/L2)
                qr = qtab[q];
                succ = (cd.y >> SW_SUCC_SHIFT) & 1u;
                const uint32_t ell = (uint32_t)(t + 1) - (cd.x & 0xFFFFu);
                atomicAdd(s_cost, (unsigned long long)((ell << 16) / (qr.y & 0xFFFFu)));   // C_k = l_k / beta, Q16 (R28); l < 2^16
                atomicAdd(&s_latsum[model], ell); atomicAdd(&s_latn[model], 1u);
                atomicAdd(&s_relkv[model], (cd.y & SW_TOK_MASK) + ((cd.y >> SW_IN_SHIFT) & SW_TOK_MASK)); atomicAdd(&s_relnrun[model], 1u);
                atomicOr(&s_occclr[2 * model + (sl >> 5)], 1u << (sl & 31));  // the slot is free from the next tick on
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
                    const uint32_t li = lbase + __popc(finm & lt_mask);
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

        // =============================================================== D-issue (R18): the new calls join the waiting list
        const uint32_t icnt = min(s_misc[1], kIssueCap);        // the executor kernel flags an overflow (err_flag)
        if (icnt) {
            const uint2 *iss = (const uint2 *)(rec + P.off_iss);
            const uint32_t nw0 = s_misc[2];
            if (nw0 + icnt > P.RCAP) { if (gl == 0) atomicOr(P.err_flag, 8u); }      // cannot happen: rcap >= 3 qcap (R9)
            else
#pragma unroll 1
                for (uint32_t j = gl; j < icnt; j += G) {
                    const uint2 r = iss[j];
                    wkey[nw0 + j] = r.x;
                    waux[nw0 + j] = make_uint2(((uint32_t)t & 0xFFFFu) | ((r.y & SW_TOK_MASK) << 16), r.y);   // issue = t, remaining = out_total
                    atomicAdd(&M_NWAIT(r.x >> 28), 1u);
                }
            g.sync();
            if (gl == 0) { s_ctr[C_ISSUED] += icnt; s_ctr[C_EXEC_DEC] += icnt; s_misc[1] = 0; s_misc[2] = nw0 + icnt; }
            g.sync();
        }

        // models that can admit (R21), judged on the state before this tick's service
        const uint32_t madm = g.ballot(gl < N && M_NWAIT(gl) > 0 && M_NRUN(gl) < s_model[gl].slots && M_KV(gl) <= s_model[gl].kv_cap);

        // =============================================================== F serve (R11): one streaming pass over the slots
        g.sync();
        {
            uint4 *hot4 = (uint4 *)hot;
            const uint32_t n_grp = P.SP >> 3;
            auto occ8_of = [&](uint32_t gi) -> uint32_t {
                const uint32_t k = s_gmodel[gi], sl0 = gi * 8 - s_sbase[k];       // first slot of the group within its model
                return (s_occ[2 * k + (sl0 >> 5)] >> (sl0 & 31)) & 0xFFu;
            };
            // Lane gl takes group gl first (its words came with the header); the non-empty groups beyond the first G are
            // compacted into a list, so that later iterations keep all lanes busy whatever the load of the pool.
            uint32_t n_list = 0;
#pragma unroll 1
            for (uint32_t g0 = G; g0 < n_grp; g0 += G) {
                const uint32_t gi = g0 + gl;
                const uint32_t o8 = gi < n_grp ? occ8_of(gi) : 0u;
                const bool ne = o8 != 0;
                const uint32_t m = g.ballot(ne);
                if (ne) s_glist[n_list + __popc(m & lt_mask)] = (uint16_t)(gi | (o8 << 8));
                n_list += __popc(m);
            }
            g.sync();
            const uint32_t n_it = 1 + (n_list + G - 1) / G;
            uint4 na = pre_a, nb = pre_b;
            uint32_t ngi = gl, nocc = gl < n_grp ? occ8_of(gl) : 0u;
#pragma unroll 1
            for (uint32_t it = 0; it < n_it; it++) {
                const uint32_t gi = ngi;
                const uint4 ha = na, hb = nb;
                const uint32_t occ8 = nocc;
                nocc = 0;
                if (it * G + gl < n_list) { const uint32_t ent = s_glist[it * G + gl]; ngi = ent & 0xFFu; nocc = ent >> 8; na = hot4[2 * ngi]; nb = hot4[2 * ngi + 1]; }
                if (occ8) {
                    const uint32_t k = s_gmodel[gi], base = s_base[k], thr = s_thr[k];
                    const Ph4 u4 = philox4x32_10_rk(gid, (uint32_t)t, gi, 0u, P.svc_rk);
                    const uint32_t uw[4] = {u4.x, u4.y, u4.z, u4.w};
                    uint32_t hh[8] = {ha.x, ha.y, ha.z, ha.w, hb.x, hb.y, hb.z, hb.w};
                    uint32_t tot = 0;
#pragma unroll
                    for (int s = 0; s < 8; s++) {
                        if ((occ8 >> s) & 1u) {
                            const uint32_t w = hh[s], rem = w & 0xFFFFu;
                            const uint32_t u16 = (s & 1) ? (uw[s >> 1] >> 16) : (uw[s >> 1] & 0xFFFFu);
                            const uint32_t tok = base + (u16 < thr ? 1u : 0u);
                            if (tok >= rem) {                                    // completes: only `rem` tokens are decoded
                                tot += rem;
                                s_clist[atomicAdd(&s_sc[0], 1u)] = (uint16_t)(gi * 8 + s);
                                hh[s] = w & 0xFFFF0000u;
                            } else {
                                tot += tok;
                                hh[s] = w - tok;
                            }
                        }
                    }
                    atomicAdd(&s_kvadd[k], tot);
                    hot4[2 * gi] = make_uint4(hh[0], hh[1], hh[2], hh[3]);
                    hot4[2 * gi + 1] = make_uint4(hh[4], hh[5], hh[6], hh[7]);
                }
            }
            g.sync();
        }

        // =============================================================== E admit (R20, R21): smallest key first, per model
        if (madm) {
            uint32_t nw = s_misc[2];
            uint32_t mleft = madm;
            // lane k tracks model k (state before this tick's service: admission precedes service, R21)
            uint32_t a_nw = 0, a_nr = 0, a_kv = 0, a_tok = 0, a_olo = 0, a_ohi = 0;
            if (gl < N) { a_nw = M_NWAIT(gl); a_nr = M_NRUN(gl); a_kv = M_KV(gl); a_olo = s_occ[2 * gl]; a_ohi = s_occ[2 * gl + 1]; }
            while (mleft) {
                if (gl < kMaxModels) s_amin[gl] = 0xFFFFFFFFu;
                if (gl == 0) s_sc[3] = 0;
                g.sync();
                // per-model minimum of the waiting keys and its list index, two admitting models per pass over the list
                // (128-bit loads, two in flight per lane).  The keys of model k are those in [k<<28, (k+1)<<28): for them,
                // and only for them, key - (k<<28) is below 2^28 - 1 in unsigned arithmetic.
                const uint4 *wk4 = (const uint4 *)wkey;
                const uint32_t n4 = (nw + 3) >> 2;
                uint32_t mscan = mleft;
#pragma unroll 1
                while (mscan) {
                    const uint32_t k0 = __ffs(mscan) - 1;
                    mscan &= mscan - 1;
                    const uint32_t k1 = mscan ? __ffs(mscan) - 1 : k0;
                    mscan &= mscan - 1;
                    const uint32_t b0 = k0 << 28, b1 = k1 << 28;
                    uint32_t d0 = 0x0FFFFFFFu, d1 = 0x0FFFFFFFu, i0 = 0, i1 = 0;
#pragma unroll 1
                    for (uint32_t j0 = 0; j0 < n4; j0 += 2 * G) {
                        const uint32_t ja = j0 + gl, jb = ja + G;
                        uint4 ka = make_uint4(~0u, ~0u, ~0u, ~0u), kb = ka;
                        if (ja < n4) ka = wk4[ja];
                        if (jb < n4) kb = wk4[jb];
                        if (ja < n4 && nw - 4 * ja < 4) { const uint32_t v = nw - 4 * ja; if (v < 2) ka.y = ~0u; if (v < 3) ka.z = ~0u; ka.w = ~0u; }
                        if (jb < n4 && nw - 4 * jb < 4) { const uint32_t v = nw - 4 * jb; if (v < 2) kb.y = ~0u; if (v < 3) kb.z = ~0u; kb.w = ~0u; }
                        const uint32_t kk[8] = {ka.x, ka.y, ka.z, ka.w, kb.x, kb.y, kb.z, kb.w};
#pragma unroll
                        for (int i = 0; i < 8; i++) {
                            const uint32_t j = ((i < 4 ? ja : jb) << 2) + (i & 3);
                            const uint32_t da = kk[i] - b0, db = kk[i] - b1;
                            if (da < d0) { d0 = da; i0 = j; }
                            if (db < d1) { d1 = db; i1 = j; }
                        }
                    }
                    const uint32_t m0 = g.umin(d0), m1 = g.umin(d1);
                    if (m0 != 0x0FFFFFFFu && d0 == m0) { s_amin[k0] = b0 + m0; s_aidx[k0] = i0; }     // keys are unique: one lane
                    if (k1 != k0 && m1 != 0x0FFFFFFFu && d1 == m1) { s_amin[k1] = b1 + m1; s_aidx[k1] = i1; }
                }
                g.sync();
                bool still = false;
                if (gl < N && ((mleft >> gl) & 1u) && s_amin[gl] != 0xFFFFFFFFu) {
                    const uint32_t k = gl, key = s_amin[k], j = s_aidx[k], id = key & 0xFFFu;
                    const uint2 wa = waux[j];
                    const uint32_t sw = wa.y, rem0 = wa.x >> 16;
                    const uint32_t need = ((sw >> SW_IN_SHIFT) & SW_TOK_MASK) + ((sw & SW_TOK_MASK) - rem0);     // R12
                    if (a_nr < s_model[k].slots && a_kv + need <= s_model[k].kv_cap) {     // else: stop at the first misfit (R21)
                        // lowest free slot of the model (R10)
                        const uint32_t sl = ~a_olo ? (uint32_t)__ffs(~a_olo) - 1u : 31u + (uint32_t)__ffs(~a_ohi);
                        if (sl < 32) a_olo |= 1u << sl; else a_ohi |= 1u << (sl - 32);
                        const uint32_t gs = s_sbase[k] + sl;
                        const uint32_t dl = P.sched_mode ? ((key >> 12) & 0xFFFFu) : (qtab[id >> 2].z & 0xFFFFu);
                        // prefill, then its first tick of service (R11)
                        const uint32_t pf = (uint32_t)(((unsigned long long)s_model[k].prefill * need) / 1000u);
                        const uint32_t usable = kDtUs - min(pf, kDtUs);
                        const uint32_t x = s_model[k].rate * usable;
                        const uint32_t bs = x / 1000000u, fr = x - bs * 1000000u;
                        const uint32_t thr = (uint32_t)(((unsigned long long)fr << 16) / 1000000u);
                        const uint32_t u16 = u16_field(draw(P, STREAM_SVC, gid, t, gs >> 3, 0), gs & 7u);
                        const uint32_t tok = min(bs + (u16 < thr ? 1u : 0u), rem0);
                        const uint32_t rem = rem0 - tok;
                        a_kv += need; a_tok += tok; a_nw -= 1; a_nr += 1;
                        hot[gs] = rem | (id << 16);
                        cold[gs] = make_uint2((wa.x & 0xFFFFu) | (dl << 16), sw);
                        if (rem == 0) s_clist[atomicAdd(&s_sc[0], 1u)] = (uint16_t)gs;
                        s_rm[atomicAdd(&s_sc[3], 1u)] = j;
                        still = a_nw > 0 && a_nr < s_model[k].slots;
                    }
                }
                mleft = g.ballot(still);
                g.sync();
                // remove the admitted entries: the holes below the new length are filled from the tail
                const uint32_t a = s_sc[3];
                if (a) {
                    const uint32_t new_len = nw - a;
                    const bool isl = gl < a;
                    const uint32_t h = isl ? s_rm[gl] : 0xFFFFFFFFu, p = new_len + gl;
                    bool tail_hole = false;
#pragma unroll 1
                    for (uint32_t x = 0; x < a; x++) tail_hole |= (g.shfl(h, (int)x) == p);
                    const bool live = isl && !tail_hole, low = isl && h < new_len;
                    const uint32_t lm = g.ballot(live), hm = g.ballot(low);
                    if (live) s_mv[__popc(lm & lt_mask)] = p;
                    g.sync();
                    if (low) { const uint32_t src = s_mv[__popc(hm & lt_mask)]; wkey[h] = wkey[src]; waux[h] = waux[src]; }
                    nw = new_len;
                    g.sync();
                }
            }
            if (gl < N) { M_NWAIT(gl) = a_nw; M_NRUN(gl) = a_nr; M_KV(gl) = a_kv + a_tok; s_occ[2 * gl] = a_olo; s_occ[2 * gl + 1] = a_ohi; }
            if (gl == 0) s_misc[2] = nw;
            g.sync();
        }
        // service totals of the requests that were RUNNING before this tick's admissions
        if (gl < N) M_KV(gl) += s_kvadd[gl];
        g.sync();

        // =============================================================== G complete: the rest of the list, then EWMA (R13)
        while (s_sc[0] > 0) flush();
        if (gl < N) {
            M_KV(gl) -= s_relkv[gl]; M_NRUN(gl) -= s_relnrun[gl];
            s_occ[2 * gl] &= ~s_occclr[2 * gl]; s_occ[2 * gl + 1] &= ~s_occclr[2 * gl + 1];
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
                const uint32_t S = s_model[k].slots, sb = s_sbase[k], cap = s_model[k].kv_cap;
                // candidates: the RUNNING requests of model k, <= 64 / G per lane; key = (deadline, id) + 1, 0 = none
                constexpr int CPL = (64 + G - 1) / G;
                uint32_t ckey[CPL], ckv[CPL];
#pragma unroll
                for (int c = 0; c < CPL; c++) {
                    const uint32_t sl = c * G + gl;
                    ckey[c] = 0; ckv[c] = 0;
                    if (sl < S && ((s_occ[2 * k + (sl >> 5)] >> (sl & 31)) & 1u)) {
                        const uint32_t h = hot[sb + sl];
                        const uint2 cd = cold[sb + sl];
                        ckey[c] = (((cd.x >> 16) << 12) | (h >> 16)) + 1u;
                        ckv[c] = ((cd.y >> SW_IN_SHIFT) & SW_TOK_MASK) + ((cd.y & SW_TOK_MASK) - (h & 0xFFFFu));
                    }
                }
                uint32_t kv = M_KV(k), npre = 0;
                const uint32_t nw_list = s_misc[2];
                while (kv > cap) {
                    uint32_t best = 0;
#pragma unroll
                    for (int c = 0; c < CPL; c++) best = max(best, ckey[c]);
                    const uint32_t wbest = g.umax(best);
                    if (wbest == 0) break;
                    uint32_t mykv = 0;
#pragma unroll
                    for (int c = 0; c < CPL; c++) {
                        if (ckey[c] == wbest) {                              // keys are unique: exactly one lane, one candidate
                            const uint32_t sl = c * G + gl, gs = sb + sl;
                            const uint32_t h = hot[gs];
                            const uint2 cd = cold[gs];
                            const uint32_t tm = P.sched_mode ? (cd.x >> 16) : (cd.x & 0xFFFFu);
                            wkey[nw_list + npre] = (k << 28) | (tm << 12) | (h >> 16);
                            waux[nw_list + npre] = make_uint2((cd.x & 0xFFFFu) | ((h & 0xFFFFu) << 16), cd.y);   // keeps progress and issue tick
                            atomicAnd(&s_occ[2 * k + (sl >> 5)], ~(1u << (sl & 31)));
                            mykv = ckv[c];
                            ckey[c] = 0;
                        }
                    }
                    kv -= g.sum(mykv);
                    npre++;
                }
                g.sync();
                if (gl == 0) { M_KV(k) = kv; M_NRUN(k) -= npre; M_NWAIT(k) += npre; s_ctr[C_PREEMPT] += npre; s_misc[2] = nw_list + npre; }
                g.sync();
            }
        }

        // =============================================================== I record (R27, R28, R33)
        IM_CONVERGE();
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
                // hard reset: live queries abandoned, pools emptied (free slots are defined by occ / the bitmaps)
                uint32_t live = 0;
#pragma unroll 1
                for (uint32_t w = gl; w < QW; w += G) live += __popc(~s_qfree[w]);
                live = g.sum(live);
                if (gl == 0) { s_ctr[C_ABANDONED] += live; s_misc[2] = 0; }
#pragma unroll 1
                for (uint32_t w = gl; w < QW; w += G) { s_qfree[w] = 0xFFFFFFFFu; s_qready[w] = 0; }
                if (gl < N) { M_NWAIT(gl) = 0; M_NRUN(gl) = 0; M_KV(gl) = 0; M_EWMA(gl) = 0; s_occ[2 * gl] = 0; s_occ[2 * gl + 1] = 0; }
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
#pragma unroll 1
            for (uint32_t b0 = 0; b0 < n_ready; b0 += G) {
                const uint32_t o = b0 + gl;
                uint32_t q = 0;
                uint4 qr = make_uint4(0, 0, 0, 0);
                if (o < n_ready) { q = find_nth(s_qready, QW, prefB, o); qr = qtab[q]; }
                emit_ready(o < n_ready, q, qr.x, qr.y >> 16, (int32_t)qr.z, t_rel);
            }
            g.sync();
            if (n_ready) {
#pragma unroll 1
                for (uint32_t w = gl; w < QW; w += G) s_qready[w] = 0;
            }
            g.sync();
        }
        // ---- A arrive (R5, R7, R8, R9)
        {
            // one Philox pass for the whole group: the last lane draws the arrival count, lane j < G - 1 draws, ahead of
            // need, the budget / input tokens of arrival j (same streams and counters as two separate passes, R2)
            const bool cnt_lane = gl == G - 1;
            const Ph4 dsp = draw(P, cnt_lane ? STREAM_ARR : STREAM_QRY, gid, t, cnt_lane ? 0u : gl, 0);
            const uint32_t xr = g.shfl(dsp.x, G - 1);
            const uint32_t *cdf = P.tab_cdf + 32u * P.env_level[e];
            uint32_t n = 0;
#pragma unroll 1
            for (uint32_t j = gl; j < 31; j += G) n += xr >= __ldg(&cdf[j]) ? 1u : 0u;
            n = g.sum(n);
            if (n) {
                const uint32_t n_free = build_prefix(g, s_qfree, QW, prefB);
                const uint32_t n_ok = min(n, n_free);
                uint32_t pidx0 = 0;
                if (gl == 0 && n_ok) pidx0 = rows_claim(P, P.plan, region, n_ok) % P.plan.regcap;
                pidx0 = g.shfl(pidx0, 0);
#pragma unroll 1
                for (uint32_t j = gl; j < n_ok; j += G) {
                    const uint32_t q = find_nth(s_qfree, QW, prefB, j);
                    const Ph4 d = j < G - 1 ? dsp : draw(P, STREAM_QRY, gid, t, j, 0);
                    const uint32_t comp = d.z < P.mix_thresh ? 0u : 1u;
                    const uint32_t budget = P.mix_lo[comp] + __umulhi(d.x, P.mix_hi[comp] - P.mix_lo[comp] + 1u);
                    const uint32_t in_tok = P.has_intok ? __ldg(&P.tab_intok[d.y >> 22]) : P.in_tok_const;
                    const int32_t dl = t + (int32_t)budget;                  // PAPER.md:117 deadline = t_arrive + beta
                    qtab[q] = make_uint4(QP_LIVE, budget | (in_tok << 16), (uint32_t)dl, (uint32_t)t);
                    P.plan.row[row_gid_wrapped(P.plan, region, pidx0, j)] = make_uint4(e, q | (t_rel << 19), (uint32_t)dl, in_tok);
                }
                g.sync();
                // the n_ok lowest free query indices are the ones taken
#pragma unroll 1
                for (uint32_t w = gl; w < QW; w += G) {
                    const uint32_t before = prefB[w], cntw = prefB[w + 1] - before;
                    if (before < n_ok) {
                        const uint32_t take = min(n_ok - before, cntw);
                        uint32_t bm = s_qfree[w];
                        if (take == cntw) bm = 0;
                    else {
#pragma unroll 1
                        for (uint32_t i = 0; i < take; i++) bm &= bm - 1;
                    }
                        s_qfree[w] = bm;
                    }
                }
                if (gl == 0) {
                    s_ctr[C_ARRIVALS] += n; s_ctr[C_DROPPED] += n - n_ok; s_ctr[C_PLANS] += n_ok;
                    s_ctr[C_SUM_LIVE_MID] += QCAP - n_free + n_ok;
                    s_misc[0] = n - n_ok;                                   // drops carried to phase I of this tick
                }
            } else {
                uint32_t live = 0;
#pragma unroll 1
                for (uint32_t w = gl; w < QW; w += G) live += __popc(~s_qfree[w]);
                live = g.sum(live);
                if (gl == 0) s_ctr[C_SUM_LIVE_MID] += live;
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
#pragma unroll 1
        for (uint32_t i = gl; i < P.hdr_words / 4; i += G) dst[i] = src[i];
    }
#undef IM_CONVERGE
#undef IM_WCONV
#undef M_NWAIT
#undef M_NRUN
#undef M_KV
#undef M_EWMA
}

void launch_sim(const Params &P, int32_t t_post, uint32_t trow_post, int32_t t_pre, uint32_t pre_mode, int32_t t0, cudaStream_t st)
{
    // G lanes per env: one lane per model in the admission and EWMA phases (N <= 16 <= G)
    static int G = 0;
    if (!G) {
        const char *ev = getenv("IM_SIM_G");
        G = ev ? atoi(ev) : 16;
        if (G != 32) G = 16;
        cudaFuncSetAttribute(k_sim<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        cudaFuncSetAttribute(k_sim<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    }
    const SimLayout L = sim_layout(P.hdr_words, P.QW, P.SP);
    const uint32_t gpb = kSimThreads / G;
    const size_t smem = (size_t)gpb * L.total;
    const uint32_t blocks = (P.E + gpb - 1) / gpb;
    if (G == 16) k_sim<16><<<blocks, kSimThreads, smem, st>>>(P, L, t_post, trow_post, t_pre, pre_mode, t0);
    else k_sim<32><<<blocks, kSimThreads, smem, st>>>(P, L, t_post, trow_post, t_pre, pre_mode, t0);
}

}  // namespace im
