// im_sim.cu — the fixed-tick simulation kernel: ONE THREAD PER ENVIRONMENT, one warp per block of 32 envs.
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
// Shape of the work.  Every phase is per-env bookkeeping driven by the few requests that change
// state in a tick, except two streaming passes: the service pass over the slots and the key scan of the admission.
// All of it runs one thread per env: the 32 lanes of a warp execute the same scalar code on 32 envs, so an
// instruction serves 32 envs where a cooperative group served one.  What makes that efficient is the layout
// (im_device.cuh): state that lanes walk in step is struct-of-arrays across the 32 envs of the block, so the service
// pass (lane l reads group g of ITS env: 32 x 16 B contiguous) and the key scan are perfectly coalesced without any
// cross-lane traffic; the header block lands in shared memory as [word][lane] by one bulk async copy (TMA) and goes
// back the same way, so its 2 x 12.5 KB cost no load / store instructions; control flow that depends on the pool only
// (slot group -> model) is uniform across the warp.  Every accumulation is an integer sum (R12, R13, R28).
//
// The service pass works on packed halves: a group of 8 slots is 8 x u16 remaining tokens in one uint4 and one Philox
// call yields the 8 sixteen-bit uniforms in the same arrangement (R2: field f = word f>>1, low half first), so two
// slots are served by a handful of packed u16x2 min / max (VIMNMX.U16x2) and plain 32-bit adds that cannot carry
// across the halves.  A free slot holds 0 and stays 0; a slot that goes from non-zero to zero has completed.
#include "im_device.cuh"

namespace im {

constexpr int kSimWarps = 2;            // 32-env blocks per CTA
constexpr int kServeWarps = 1;            // one (block, model) unit per CTA: 32 single-warp CTAs per SM turn over faster than 4 x 8 warps (0.0879 -> 0.0811 ms)
constexpr uint32_t kFull = 0xffffffffu;

// per-warp dynamic shared memory of k_sim: the header [hdr_words][32], one bulk copy in, one out.  Shared memory is what
// limits the resident warps of this latency-bound kernel, so the completion bytes and token counts of k_serve (read once,
// in lane order) stay in global memory
struct SimSmem { uint32_t hdr_bytes, per_warp; };
static SimSmem sim_smem(const Params &P)
{
    SimSmem L;
    L.hdr_bytes = P.hdr_words * 128u;
    L.per_warp = L.hdr_bytes;
    return L;
}

__device__ __forceinline__ uint32_t vmin2(uint32_t a, uint32_t b) { return __vminu2(a, b); }   // VIMNMX.U16x2
__device__ __forceinline__ uint32_t vmax2(uint32_t a, uint32_t b) { return __vmaxu2(a, b); }

// Two slots of a group for one tick (R11).  r = remaining tokens (two u16), u = their uniforms (two u16),
// base2 / thr2 = the model's base tokens and Bernoulli threshold in both halves.  Returns the new remaining tokens;
// adds the decoded tokens to totp (packed) and the completion flags (bit 0 / bit 16) shifted by `j` to cacc.
__device__ __forceinline__ uint32_t serve_pair(uint32_t r, uint32_t u, uint32_t base2, uint32_t thr2, int j, uint32_t &totp, uint32_t &cacc)
{
    const uint32_t e2 = vmin2(vmax2(u, thr2) - u, 0x00010001u);     // u16 < thr per half: max(u, thr) - u is non-zero iff u < thr
    const uint32_t dec = vmin2(base2 + e2, r);                      // tokens decoded: capped by what remains (0 for a free slot)
    const uint32_t rn = r - dec;                                    // no borrow: dec <= r in both halves
    totp += dec;
    cacc += (vmin2(r, 0x00010001u) - vmin2(rn, 0x00010001u)) << j;  // non-zero -> zero: completed
    return rn;
}

// sixteen-bit field f (0..7) of a Philox output (R2: word f>>1, low half first)
__device__ __forceinline__ uint32_t u16_field(const Ph4 &u, uint32_t f)
{
    const uint32_t w = (f >> 1) == 0 ? u.x : ((f >> 1) == 1 ? u.y : ((f >> 1) == 2 ? u.z : u.w));
    return (f & 1u) ? (w >> 16) : (w & 0xFFFFu);
}

// =================================================================================================== F serve (R11)
// The service pass of tick t: one streaming pass over the slots of every env.  It needs nothing but `hot` (a free slot
// holds 0), so it is a kernel of its own with no shared memory and all its loads in flight at once: a warp takes the
// (<= 8) slot groups of ONE model of one 32-env block, lane = env, so every load / store is 512 contiguous bytes and
// the model's parameters are uniform.  Results for k_sim: the tokens decoded per (env, model) and one completion byte
// per (env, group) (bits 0-3 = slots 0, 2, 4, 6; bits 4-7 = slots 1, 3, 5, 7), both SoA-32 behind the header.
// The requests admitted in THIS tick are served by k_sim's admission phase (prefill, R11): they are not in `hot` yet.
__global__ void __launch_bounds__(kServeWarps * 32, 32)
k_serve(const Params P, int32_t t)
{
    griddep_wait();
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t w = blockIdx.x * kServeWarps + (threadIdx.x >> 5);
    if (w >= P.NB * P.N) return;
    const uint32_t blk = w / P.N, k = w % P.N;     // ascending: k_sim walks the blocks in descending order, so the blocks it starts with are the ones this kernel wrote last (still in L2)
    const uint32_t g0 = P.slot_base[k] >> 3, ng = (P.slot_base[k + 1] - P.slot_base[k]) >> 3;    // 1 .. 8 groups
    const uint32_t gid = P.env_id_base + blk * 32u + lane;
    uint8_t *blkp = P.env_base + (size_t)blk * P.blk_stride;
    uint4 *hot4 = reinterpret_cast<uint4 *>(blkp + P.off_hot) + lane;                   // group g at hot4[g * 32]
    uint8_t *cmb = blkp + P.off_cm + lane * 4u;                                         // byte of group g at cmb[(g >> 2) * 128 + (g & 3)]
    const uint32_t x = P.model[k].rate * kDtUs;                                         // rate <= 80000 => fits 32 bits
    const uint32_t base2 = (x / 1000000u) * 0x00010001u;
    const uint32_t thr2 = (uint32_t)(((unsigned long long)(x % 1000000u) << 16) / 1000000u) * 0x00010001u;   // R11: Bernoulli to 2^-16
    uint4 h[8];
#pragma unroll
    for (int i = 0; i < 8; i++) if ((uint32_t)i < ng) h[i] = hot4[(g0 + i) * 32u];
    uint32_t tot = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) {
        if ((uint32_t)i < ng) {
            const uint32_t g = g0 + i;
            const bool any = (h[i].x | h[i].y | h[i].z | h[i].w) != 0;
            uint32_t cacc = 0;
            if (__any_sync(kFull, any)) {
                const Ph4 u = philox4x32_10_rk(gid, (uint32_t)t, g, 0u, P.svc_rk);
                uint32_t totp = 0;
                uint4 r;
                r.x = serve_pair(h[i].x, u.x, base2, thr2, 0, totp, cacc);
                r.y = serve_pair(h[i].y, u.y, base2, thr2, 1, totp, cacc);
                r.z = serve_pair(h[i].z, u.z, base2, thr2, 2, totp, cacc);
                r.w = serve_pair(h[i].w, u.w, base2, thr2, 3, totp, cacc);
                tot += (totp & 0xFFFFu) + (totp >> 16);
                if (any) hot4[g * 32u] = r;
            }
            cmb[(g >> 2) * 128u + (g & 3u)] = (uint8_t)((cacc & 0xFu) | ((cacc >> 12) & 0xF0u));
        }
    }
    reinterpret_cast<uint32_t *>(blkp + P.off_kvt)[k * 32u + lane] = tot;
}

// tick arguments: t_post < 0 => no post phases; pre_mode 0 none, 1 full (A, B, rows), 2 snapshot only
__global__ void __launch_bounds__(kSimWarps * 32, 8)
k_sim(const Params P, const SimSmem L, int32_t t_post, uint32_t trow_post, int32_t t_pre, uint32_t pre_mode, int32_t t0)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ uint64_t s_bar[kSimWarps];
    __shared__ uint32_t s_rate[kMaxModels], s_slots[kMaxModels], s_kvcap[kMaxModels], s_prefill[kMaxModels];
    __shared__ uint32_t s_sbase[kMaxModels + 1];
    __shared__ float s_kvinv[kMaxModels];
    __shared__ uint8_t s_gmodel[128];                                       // group of 8 slots -> model
    const uint32_t lane = threadIdx.x & 31u, wib = threadIdx.x >> 5;
    if (threadIdx.x < P.N) {
        const ModelTab m = P.model[threadIdx.x];
        s_rate[threadIdx.x] = m.rate; s_slots[threadIdx.x] = m.slots; s_kvcap[threadIdx.x] = m.kv_cap; s_prefill[threadIdx.x] = m.prefill;
        s_kvinv[threadIdx.x] = m.kv_inv;
    }
    if (threadIdx.x <= kMaxModels) s_sbase[threadIdx.x] = P.slot_base[threadIdx.x];
    for (uint32_t g = threadIdx.x; g < P.n_grp; g += blockDim.x) {
        uint32_t k = 0;
        while (P.slot_base[k + 1] <= g * 8) k++;
        s_gmodel[g] = (uint8_t)k;
    }
    if (lane == 0) bulk::mbar_init(&s_bar[wib], 1);
    bulk::fence_mbar_init();
    __syncthreads();
    griddep_wait();                                                         // everything above reads the spec only
    // blocks in descending order: neutral in general; where load rises with the env index (the utilisation sweep of
    // configs[3]-[4]) the heaviest blocks start first and the last wave is the lightest
    const uint32_t wg = blockIdx.x * kSimWarps + wib;
    if (wg >= P.NB) return;
    const uint32_t blk = P.NB - 1u - wg;
    const uint32_t e = blk * 32u + lane;
    const bool active = e < P.E;
    const uint32_t gid = P.env_id_base + e;
    const uint32_t N = P.N, QW = P.QW;
    const uint32_t region = blk % P.n_regions;
    const uint32_t lt_mask = (1u << lane) - 1u;

    unsigned char *sm = smem_raw + (size_t)wib * L.per_warp;
    uint32_t *s_hdr = reinterpret_cast<uint32_t *>(sm) + lane;                          // word w at s_hdr[w * 32]
#define H(w) s_hdr[(w) * 32u]
#define M_W0(k) s_hdr[(3u * (k)) * 32u]            /* n_wait | n_run << 16 */
#define M_KV(k) s_hdr[(3u * (k) + 1u) * 32u]
#define M_EWMA(k) s_hdr[(3u * (k) + 2u) * 32u]
#define OCC(w) s_hdr[(P.hw_occ + (w)) * 32u]       /* bit gs = global slot gs taken */
#define QFREE(w) s_hdr[(P.hw_qfree + (w)) * 32u]
#define NEXTW(c) s_hdr[(P.hw_next + ((c) >> 2)) * 32u]    /* next[c]: byte c & 3 */
#define HEADW(k) s_hdr[(P.hw_head + ((k) >> 2)) * 32u]    /* head[k]: byte k & 3 */

    uint8_t *blkp = P.env_base + (size_t)blk * P.blk_stride;
    if (lane == 0) {
        bulk::mbar_expect_tx(&s_bar[wib], L.hdr_bytes);
        bulk::g2s(sm, blkp, L.hdr_bytes, &s_bar[wib]);
    }
    uint4 *hot4 = reinterpret_cast<uint4 *>(blkp + P.off_hot) + lane;                   // group g at hot4[g * 32]
    uint16_t *hot16 = reinterpret_cast<uint16_t *>(blkp + P.off_hot) + lane * 8u;       // slot gs at hot16[(gs >> 3) * 256 + (gs & 7)]
    uint32_t *wkey = reinterpret_cast<uint32_t *>(blkp + P.off_wkey + (size_t)lane * P.wkey_stride);   // entry i of chunk c at [c * 16 + i]
    uint4 *cold = reinterpret_cast<uint4 *>(blkp + P.off_cold + (size_t)lane * P.cold_stride);
    uint2 *waux = reinterpret_cast<uint2 *>(blkp + P.off_waux + (size_t)lane * P.waux_stride);
    uint4 *qtab = reinterpret_cast<uint4 *>(blkp + P.off_q + (size_t)lane * P.q_stride);
    uint32_t *qready = reinterpret_cast<uint32_t *>(blkp + P.off_qready) + lane;        // word w at qready[w * 32]
    uint32_t *ctr = reinterpret_cast<uint32_t *>(blkp + P.off_ctr) + lane;              // counter c at ctr[c * 32]
    uint32_t *cmg = reinterpret_cast<uint32_t *>(blkp + P.off_cm) + lane;               // completion bytes of the tick (k_serve): word w at cmg[w * 32]

    // The arrival count of tick t_pre (R5) depends on nothing but (env, tick): one Philox call and a binary search of
    // the level's CDF row (count = #{j < 31 : x >= cdf[j]}; the row is monotone, so it is the first j with x < cdf[j]).
    // Done here, its loads overlap the header's flight.
    uint32_t n_arr_pre = 0;
    if (pre_mode == 1 && active) {
        const uint32_t xr = draw(P, STREAM_ARR, gid, t_pre, 0u, 0).x;
        const uint32_t *cdf = P.tab_cdf + 32u * P.env_level[e];
        uint32_t lo = 0, hi = 31;
#pragma unroll
        for (int s = 0; s < 5; s++) {
            const uint32_t mid = (lo + hi) >> 1;
            if (lo < hi) { if (xr >= __ldg(&cdf[mid])) lo = mid + 1; else hi = mid; }
        }
        n_arr_pre = lo;
    }
    // counters of this launch (named registers: every site is static)
    uint32_t c_arr = 0, c_drop = 0, c_fin = 0, c_solved = 0, c_missed = 0, c_issued = 0, c_done = 0, c_preempt = 0, c_soj = 0,
             c_live = 0, c_plans = 0, c_run = 0, c_wait = 0, c_aband = 0;

    // one warp-aggregated claim of executor rows: lanes with nc > 0 (<= 3) get consecutive ring positions of the region
    auto claim_exec_rows = [&](uint32_t nc, uint32_t &idx0) -> bool {
        const uint32_t b0 = __ballot_sync(kFull, (nc & 1u) != 0), b1 = __ballot_sync(kFull, (nc & 2u) != 0);
        const uint32_t tot = __popc(b0) + 2u * __popc(b1);
        if (tot == 0) return false;
        uint32_t base = 0;
        if (lane == 0) base = rows_claim(P, P.exec, region, tot) % P.exec.regcap;
        idx0 = __shfl_sync(kFull, base, 0) + __popc(b0 & lt_mask) + 2u * __popc(b1 & lt_mask);
        if (idx0 >= P.exec.regcap) idx0 -= P.exec.regcap;
        return true;
    };
    // the (<= 64) occupancy bits of the model whose slots start at global slot sb (a multiple of 8): bit s = slot s
    auto occ_window = [&](uint32_t sb, uint32_t &olo, uint32_t &ohi) {
        const uint32_t w = sb >> 5, sh = sb & 31u;
        const uint32_t a = OCC(w), b = OCC(w + 1u), c = OCC(w + 2u);     // two padding words follow the bitmap
        olo = __funnelshift_r(a, b, sh); ohi = __funnelshift_r(b, c, sh);
    };
    // ---- waiting lists: one unordered list per model, a linked list of 32-entry chunks of a per-env pool (im_device.cuh).
    // Only the HEAD chunk of a model is partly filled: with n entries it holds ((n - 1) & 31) + 1 of them.
    auto byte_get = [](uint32_t w, uint32_t i) { return (w >> (8u * (i & 3u))) & 0xFFu; };
    auto byte_put = [](uint32_t w, uint32_t i, uint32_t v) { const uint32_t sh = 8u * (i & 3u); return (w & ~(0xFFu << sh)) | (v << sh); };
    uint32_t free_head = 0xFFu;                                  // head of the free-chunk list (kept in misc0 between launches)
    // insert: into the head chunk if it has room, else into a fresh chunk that becomes the head.  A fresh chunk is written
    // whole (its key and 31 x 0xFFFFFFFF = one full 128-byte line): a full-line write needs no fill read from DRAM, and the
    // partial stores of the keys that follow in this tick merge into it in the L2 (measured: 0.299 ms per tick against
    // 0.305 with a lone 16-byte store).  Entries are valid up to the list's count and scans read only those units.
    auto list_insert = [&](uint32_t k, uint32_t key, uint2 aux) {
        const uint32_t w0 = M_W0(k), n = w0 & 0xFFFFu;
        uint32_t c = byte_get(HEADW(k), k), pos = n & (kChunk - 1u);
        if (pos == 0) {                                          // empty list or full head chunk
            const uint32_t nc = free_head;                       // the pool always has a free chunk here (rcap >= 3 qcap, R9)
            free_head = byte_get(NEXTW(nc), nc);
            NEXTW(nc) = byte_put(NEXTW(nc), nc, n ? c : 0xFFu);
            HEADW(k) = byte_put(HEADW(k), k, nc);
            c = nc;
            uint4 *ck = reinterpret_cast<uint4 *>(wkey + c * kChunk);
            ck[0] = make_uint4(key, ~0u, ~0u, ~0u);
#pragma unroll
            for (int i = 1; i < (int)kChunk / 4; i++) ck[i] = make_uint4(~0u, ~0u, ~0u, ~0u);
        } else {
            wkey[c * kChunk + pos] = key;
        }
        waux[c * kChunk + pos] = aux;
        M_W0(k) = w0 + 1u;
    };
    // smallest key of model k (n entries): walk its chunks (the lanes of a warp walk theirs in step, so their loads go out
    // together), reading only the units that hold entries: the head chunk is the only one partly filled.
    // Returns the key and the 4-entry unit that holds it
    auto list_min = [&](uint32_t k, uint32_t n, uint32_t &bkey, uint32_t &bunit) {
        bkey = ~0u; bunit = 0;
        uint32_t c = byte_get(HEADW(k), k), nu = (((n - 1u) & (kChunk - 1u)) >> 2) + 1u;
#pragma unroll 1
        while (c != 0xFFu) {
            const uint4 *ck = reinterpret_cast<const uint4 *>(wkey + c * kChunk);
            uint4 v[kChunk / 4];
#pragma unroll
            for (int i = 0; i < (int)kChunk / 4; i++) v[i] = (uint32_t)i < nu ? ck[i] : make_uint4(~0u, ~0u, ~0u, ~0u);
            const uint32_t cn = byte_get(NEXTW(c), c);
#pragma unroll
            for (int i = 0; i < (int)kChunk / 4; i++) {
                const uint32_t m = min(min(v[i].x, v[i].y), min(v[i].z, v[i].w));
                if (m < bkey) { bkey = m; bunit = c * (kChunk / 4) + i; }
            }
            c = cn; nu = kChunk / 4;
        }
    };
    // remove entry j (= chunk * 32 + position) of model k: the last entry of the head chunk fills the hole; `lk` / `la`
    // are that entry's key and aux word, fetched by the caller ahead of time
    auto list_remove = [&](uint32_t k, uint32_t j, uint32_t lk, uint2 la) {
        const uint32_t w0 = M_W0(k), n = w0 & 0xFFFFu;
        const uint32_t h = byte_get(HEADW(k), k), lp = (n - 1u) & (kChunk - 1u), lj = h * kChunk + lp;
        if (lj != j) { wkey[j] = lk; waux[j] = la; }
        wkey[lj] = ~0u;
        if (lp == 0) {                                           // the head chunk is empty: back to the pool
            const uint32_t nx = byte_get(NEXTW(h), h);
            HEADW(k) = byte_put(HEADW(k), k, nx);
            NEXTW(h) = byte_put(NEXTW(h), h, free_head);
            free_head = h;
        }
        M_W0(k) = w0 - 1u;
    };

    if (t_post >= 0) {
        const int32_t t = t_post;
        const uint32_t done = (P.episode_ticks && ((uint32_t)(t + 1) % P.episode_ticks) == 0) ? 1u : 0u;
        const bool emit = (pre_mode == 1) && !done;
        const uint32_t t_rel_next = (uint32_t)(t + 1 - t0);

        // the first four issue records, fetched before their count is known (it sits in the header still in flight)
        const uint2 *iss = reinterpret_cast<const uint2 *>(blkp + P.off_iss) + lane;
        uint2 r[4];
#pragma unroll
        for (uint32_t i = 0; i < 4; i++) r[i] = iss[i * 32u];
        bulk::mbar_wait(&s_bar[wib], 0);

        // A WAITING request of model k (key, aux word wa, KV need) becomes RUNNING (R10, R11): lowest free slot of the model,
        // prefill, its first tick of service, the slot's record.  w0 / kv = the model's counts before; returns the tokens of
        // the first tick (the caller adds them to kv_used when admission is over for the model: R21 judges on the state
        // before the tick's service).  n_run < S_k is the caller's check.
        auto place = [&](uint32_t k, uint32_t key, uint2 wa, uint32_t need, uint32_t w0, uint32_t kv) -> uint32_t {
            const uint32_t sw = wa.y, rem0 = wa.x >> 16, id = key & 0xFFFu;
            uint32_t olo, ohi;
            occ_window(s_sbase[k], olo, ohi);
            const uint32_t sl = ~olo ? (uint32_t)__ffs(~olo) - 1u : 31u + (uint32_t)__ffs(~ohi);   // lowest free slot (R10): n_run < S_k, so it is one of the model's
            const uint32_t gs = s_sbase[k] + sl;
            OCC(gs >> 5) |= 1u << (gs & 31u);
            const uint32_t dl = P.sched_mode ? ((key >> 12) & 0xFFFFu) : (qtab[id >> 2].z & 0xFFFFu);
            // prefill, then its first tick of service (R11)
            // (32-bit arithmetic throughout: prefill * need <= 5e7 by the spec check "prefill is sub-tick",
            // rate * usable <= 4e9, and fr * 2^16 / 10^6 = fr * 1024 / 15625 exactly, fr * 1024 < 2^30)
            const uint32_t pf = (s_prefill[k] * need) / 1000u;
            const uint32_t usable = kDtUs - min(pf, kDtUs);
            const uint32_t x = s_rate[k] * usable;
            const uint32_t bs = x / 1000000u, fr = x - bs * 1000000u;
            const uint32_t thr = (fr * 1024u) / 15625u;
            const uint32_t u16 = u16_field(philox4x32_10_rk(gid, (uint32_t)t, gs >> 3, 0u, P.svc_rk), gs & 7u);
            const uint32_t tok = min(bs + (u16 < thr ? 1u : 0u), rem0);
            const uint32_t rem = rem0 - tok;
            hot16[(gs >> 3) * 256u + (gs & 7u)] = (uint16_t)rem;
            st256(&cold[2u * gs], make_uint4((wa.x & 0xFFFFu) | (dl << 16), sw, id, 0u), make_uint4(0u, 0u, 0u, 0u));
            if (rem == 0) {
                const uint32_t g = gs >> 3;
                cmg[(g >> 2) * 32u] |= 1u << (8u * (g & 3u) + ((gs & 7u) >> 1) + 4u * (gs & 1u));   // the lane's own word; rare
            }
            M_W0(k) = w0 + 0x10000u;                              // n_run++
            M_KV(k) = kv + need;
            return tok;
        };

        // =============================================================== D-issue (R18): the new calls join the waiting list -
        // or skip it.  A call that is the model's ONLY issue of the tick and finds the model's queue empty is exactly what
        // the admission phase would look at first for that model, alone: if a slot is free and its KV fits it is admitted
        // here, straight from the issue record, and the list (two stores now, two loads and a store in the admission
        // phase, all at data-dependent addresses) is never touched; if not, it waits like any other.  Below saturation
        // that is most calls.  (Decided only when all of the tick's issue records are the four already in registers.)
        const uint32_t drops_in = H(P.hw_misc) & 0xFFFFu;        // R9: drops of this tick's phase A
        free_head = H(P.hw_misc) >> 16;
        {
            uint32_t icnt = H(P.hw_misc + 1u);
            if (icnt > kIssueCap) icnt = kIssueCap;              // the executor kernel flags the overflow (err_flag)
            uint32_t queued = ~0u;                                // models whose issues must go through the list
            if (icnt <= 4u) {
                uint32_t seen = 0;
                queued = 0;
#pragma unroll
                for (uint32_t i = 0; i < 4; i++)
                    if (i < icnt) { const uint32_t b = 1u << (r[i].x >> 28); queued |= seen & b; seen |= b; }
            }
#pragma unroll 1
            for (uint32_t j0 = 0; j0 < icnt; j0 += 4) {            // four records in flight per lane
                if (j0) {
#pragma unroll
                    for (uint32_t i = 0; i < 4; i++) if (j0 + i < icnt) r[i] = iss[(j0 + i) * 32u];
                }
#pragma unroll 1
                for (uint32_t i = 0; i < 4 && j0 + i < icnt; i++) {
                    const uint2 rec = i == 0 ? r[0] : (i == 1 ? r[1] : (i == 2 ? r[2] : r[3]));
                    const uint32_t k = rec.x >> 28;
                    const uint2 aux = make_uint2(((uint32_t)t & 0xFFFFu) | ((rec.y & SW_TOK_MASK) << 16), rec.y);   // issue = t, remaining = out_total
                    bool direct = false;
                    if (!((queued >> k) & 1u)) {
                        const uint32_t w0 = M_W0(k), kv = M_KV(k);
                        const uint32_t need = (rec.y >> SW_IN_SHIFT) & SW_TOK_MASK;                          // R12: nothing decoded yet
                        if ((w0 & 0xFFFFu) == 0 && (w0 >> 16) < s_slots[k] && kv + need <= s_kvcap[k]) {
                            M_KV(k) += place(k, rec.x, aux, need, w0, kv);
                            direct = true;
                        }
                    }
                    if (!direct) list_insert(k, rec.x, aux);
                }
            }
            c_issued += icnt;
        }

        // =============================================================== E admit (R20, R21): smallest key first, per model.
        // Judged on the state before this tick's service (admission precedes service): the tokens the admitted requests
        // decode in their first tick are added when the lane is done with the model, the tokens of k_serve after the phase.
        {
            uint32_t madm = 0;
#pragma unroll 1
            for (uint32_t k = 0; k < N; k++) {
                const uint32_t w0 = M_W0(k);
                if ((w0 & 0xFFFFu) > 0 && (w0 >> 16) < s_slots[k] && M_KV(k) <= s_kvcap[k]) madm |= 1u << k;
            }
            uint32_t tokacc = 0;
#pragma unroll 1
            while (__any_sync(kFull, madm != 0)) {
                if (madm) {
                    const uint32_t k = (uint32_t)__ffs(madm) - 1u;
                    const uint32_t n0 = M_W0(k) & 0xFFFFu, hc = byte_get(HEADW(k), k);
                    uint32_t key, j = 0, lk;
                    uint2 wa = make_uint2(0, 0), la;
                    if (n0 <= 4u) {
                        // a short queue (the usual case below saturation) is the first n0 entries of its head chunk: keys and
                        // aux words come in ONE round trip (entries beyond n0 hold 0xFFFFFFFF)
                        const uint4 ku = *reinterpret_cast<const uint4 *>(wkey + hc * kChunk);
                        const uint4 a01 = *reinterpret_cast<const uint4 *>(waux + hc * kChunk), a23 = *reinterpret_cast<const uint4 *>(waux + hc * kChunk + 2);
                        uint32_t p = 0;
                        key = ku.x;
                        if (ku.y < key) { key = ku.y; p = 1; }
                        if (ku.z < key) { key = ku.z; p = 2; }
                        if (ku.w < key) { key = ku.w; p = 3; }
                        j = hc * kChunk + p;
                        wa = p == 0 ? make_uint2(a01.x, a01.y) : (p == 1 ? make_uint2(a01.z, a01.w) : (p == 2 ? make_uint2(a23.x, a23.y) : make_uint2(a23.z, a23.w)));
                        const uint32_t lp = n0 - 1u;             // the entry that fills the hole: the last one
                        lk = lp == 0 ? ku.x : (lp == 1 ? ku.y : (lp == 2 ? ku.z : ku.w));
                        la = lp == 0 ? make_uint2(a01.x, a01.y) : (lp == 1 ? make_uint2(a01.z, a01.w) : (lp == 2 ? make_uint2(a23.x, a23.y) : make_uint2(a23.z, a23.w)));
                    } else {
                        // the entry that will fill the hole if the head of the queue is admitted (last of the head chunk):
                        // its address is known now, so it is fetched together with the keys
                        const uint32_t lj = hc * kChunk + ((n0 - 1u) & (kChunk - 1u));
                        lk = wkey[lj];
                        la = waux[lj];
                        uint32_t bunit;
                        list_min(k, n0, key, bunit);
                        if (key != ~0u) {
                            // position of the key inside its unit (keys are unique)
                            const uint4 bu = *reinterpret_cast<const uint4 *>(wkey + bunit * 4u);
                            j = bunit * 4u + (bu.x == key ? 0u : (bu.y == key ? 1u : (bu.z == key ? 2u : 3u)));
                            wa = waux[j];
                        }
                    }
                    bool again = false;
                    if (key != ~0u) {
                        const uint32_t sw = wa.y, rem0 = wa.x >> 16;
                        const uint32_t need = ((sw >> SW_IN_SHIFT) & SW_TOK_MASK) + ((sw & SW_TOK_MASK) - rem0);     // R12
                        const uint32_t w0 = M_W0(k), nr = w0 >> 16, kv = M_KV(k), slots = s_slots[k];
                        if (nr < slots && kv + need <= s_kvcap[k]) {                          // else: stop at the first misfit (R21)
                            tokacc += place(k, key, wa, need, w0, kv);
                            list_remove(k, j, lk, la);
                            again = (w0 & 0xFFFFu) > 1u && nr + 1u < slots;
                        }
                    }
                    if (!again) { madm &= madm - 1u; M_KV(k) += tokacc; tokacc = 0; }
                }
            }
        }
        // F serve ran in k_serve.  Its results - tokens per model, one completion byte per slot group - are fetched here
        // in one round trip (lane order: coalesced): admission is judged on the state before the tick's service, and up
        // to here the registers belong to the admission phase.
        constexpr uint32_t kCmBatch = 16;                        // completion words held in registers at a time (64 slot groups)
        uint32_t cw[kCmBatch];
        {
            uint32_t kvt[kMaxModels];
            const uint32_t *kvs = reinterpret_cast<const uint32_t *>(blkp + P.off_kvt) + lane;
#pragma unroll
            for (uint32_t k = 0; k < kMaxModels; k++) kvt[k] = k < N ? kvs[k * 32u] : 0u;
#pragma unroll
            for (uint32_t i = 0; i < kCmBatch; i++) cw[i] = i < P.cm_words ? cmg[i * 32u] : 0u;
#pragma unroll
            for (uint32_t k = 0; k < kMaxModels; k++) if (k < N) M_KV(k) += kvt[k];
        }

        // =============================================================== G complete (R1, R13, R27, R28): completion bits in
        // slot order = model order, so the per-model latency mean of the EWMA (R13) is a run-length accumulation.
        // A three-stage software pipeline per lane hides the two dependent loads of a completion (the slot's cold word,
        // then the plan word of its query): while completion i is processed, the query of i+1 and the cold word of i+2
        // are in flight.  Rows / log records are claimed with one atomic each and written one iteration later, so the
        // claim's round trip overlaps the next completion instead of stalling this one.
        uint32_t rew = 0, miss = 0;
        unsigned long long cost = 0;
        {
            uint32_t wb = 0, wi = 0, wmask = 0, bits = 0, curk = ~0u, latsum = 0, latn = 0;
            auto ewma_flush = [&]() {
                if (curk != ~0u && latn > 0) {
                    const int32_t mean_q8 = (int32_t)((latsum << 8) / latn);
                    int32_t ew = (int32_t)M_EWMA(curk);
                    ew += (mean_q8 - ew) >> 3;
                    M_EWMA(curk) = (uint32_t)ew;
                }
            };
            // next completion bit of this lane: global slot, or ~0u
            auto next_slot = [&]() -> uint32_t {
                if (bits == 0) {                                  // next non-zero word of the batch (a select chain: registers)
                    if (wmask == 0) return ~0u;
                    wi = (uint32_t)__ffs(wmask) - 1u;
                    wmask &= wmask - 1u;
#pragma unroll
                    for (uint32_t i = 0; i < kCmBatch; i++) bits = wi == i ? cw[i] : bits;
                }
                const uint32_t b = (uint32_t)__ffs(bits) - 1u;
                bits &= bits - 1u;
                const uint32_t g = (wb + wi) * 4u + (b >> 3), bb = b & 7u;
                return g * 8u + (((bb & 3u) << 1) | (bb >> 2));
            };
            // Log records and executor rows of the tick are buffered per lane (two of each; more than that is rare and
            // claims for itself) and written after the loop with ONE claim per warp each: a claim is an atomic on the
            // region's counter, and 32 lanes x several events per tick on the same line queue up in the L2
            uint32_t nf = 0, nr = 0;                              // buffered finalisations / ready queries of this lane
            uint4 f_rec[2];
            uint32_t r_q[2], r_pw[2], r_io[2], r_dl[2];          // ready: query, plan word (stage to dispatch), in_tok, deadline
            auto emit_rows = [&](uint32_t idx, uint32_t q, uint32_t pw, uint32_t in_tok, uint32_t dl) {
                uint32_t a0, nc;
                stage_calls((pw >> 2) & 3u, (pw >> 6) & 7u, (pw >> 9) & 7u, a0, nc);
                write_exec_rows(P, region, idx % P.exec.regcap, e, q, pw, in_tok, (int32_t)dl, t_rel_next, a0, nc);
            };
#pragma unroll 1
            for (wb = 0; wb < P.cm_words; wb += kCmBatch) {       // one pass unless the pool has more than 512 slots
                if (wb) {
#pragma unroll
                    for (uint32_t i = 0; i < kCmBatch; i++) cw[i] = wb + i < P.cm_words ? cmg[(wb + i) * 32u] : 0u;
                }
                wmask = 0; bits = 0;
#pragma unroll
                for (uint32_t i = 0; i < kCmBatch; i++) wmask |= cw[i] ? 1u << i : 0u;
                uint32_t gs0 = next_slot(), gs1 = ~0u, gs2 = ~0u;
                uint4 cd0 = make_uint4(0, 0, 0, 0), cd1 = cd0, cd2 = cd0, qr0 = cd0, qr1 = cd0;
                if (gs0 != ~0u) { cd0 = cold[2u * gs0]; gs1 = next_slot(); }
                if (gs1 != ~0u) cd1 = cold[2u * gs1];
                if (gs0 != ~0u) qr0 = qtab[cd0.z >> 2];
#pragma unroll 1
                while (gs0 != ~0u) {
                    if (gs1 != ~0u) { gs2 = next_slot(); if (gs2 != ~0u) cd2 = cold[2u * gs2]; qr1 = qtab[cd1.z >> 2]; }
                    else gs2 = ~0u;
                    // ---- completion of the request in slot gs0
                    const uint32_t k = s_gmodel[gs0 >> 3];
                    const uint32_t q = cd0.z >> 2;                                  // id = 4 q + agent
                    const uint32_t ell = (uint32_t)(t + 1) - (cd0.x & 0xFFFFu);
                    cost += (unsigned long long)((ell << 16) / (qr0.y & 0xFFFFu));  // C_k = l_k / beta, Q16 (R28); l < 2^16
                    if (k != curk) { ewma_flush(); curk = k; latsum = 0; latn = 0; }
                    latsum += ell; latn++;
                    M_W0(k) -= 0x10000u;                                            // n_run--
                    M_KV(k) -= (cd0.y & SW_TOK_MASK) + ((cd0.y >> SW_IN_SHIFT) & SW_TOK_MASK);
                    OCC(gs0 >> 5) &= ~(1u << (gs0 & 31u));
                    c_done++;
                    uint32_t pw = qr0.x;
                    const uint32_t pend = ((pw >> QP_PEND_SHIFT) & 3u) - 1u;
                    pw = (pw & ~(3u << QP_PEND_SHIFT)) | (pend << QP_PEND_SHIFT) | (((cd0.y >> SW_SUCC_SHIFT) & 1u) << QP_SUCC_SHIFT);   // R19: OR
                    bool fin = false, ready = false;
                    if (pend == 0) { if (((pw >> 9) & 7u) == ((pw >> 12) & 7u)) fin = true; else ready = true; }
                    if (fin) {
                        // finalise (R27): reward, SLO miss, sojourn, query log
                        const uint32_t solved = (pw >> QP_SUCC_SHIFT) & 1u;
                        const uint32_t sojourn = (uint32_t)(t + 1 - (int32_t)qr0.w);
                        const uint32_t late = (t + 1 > (int32_t)qr0.z) ? 1u : 0u;
                        rew += solved; miss += late;
                        c_fin++; c_solved += solved; c_missed += late; c_soj += sojourn;
                        const uint4 rec = make_uint4(gid, qr0.w, sojourn, (qr0.y & 0xFFFFu) | (solved << 16) | (((pw >> 2) & 3u) << 17) | (((pw >> 6) & 7u) << 19));
                        if (nf == 0) f_rec[0] = rec;
                        else if (nf == 1) f_rec[1] = rec;
                        else {
                            const uint32_t li = atomicAdd(&P.qlog.cnt[region * kCntStride], 1u);
                            if (li + 1u > P.qlog.regcap) atomicOr(P.err_flag, 2u);
                            P.qlog.rec[(size_t)region * P.qlog.regcap + (li % P.qlog.regcap)] = rec;
                        }
                        nf++;
                        QFREE(q >> 5) |= 1u << (q & 31u);
                    } else if (ready && emit) {
                        // next stage of a query whose calls all completed (R17): executor rows of tick t + 1;
                        // stage++, pending = nc: the calls are issued in phase D of the coming tick
                        uint32_t a0, nc;
                        stage_calls((pw >> 2) & 3u, (pw >> 6) & 7u, (pw >> 9) & 7u, a0, nc);
                        if (nr == 0) { r_q[0] = q; r_pw[0] = pw; r_io[0] = qr0.y >> 16; r_dl[0] = qr0.z; }
                        else if (nr == 1) { r_q[1] = q; r_pw[1] = pw; r_io[1] = qr0.y >> 16; r_dl[1] = qr0.z; }
                        else emit_rows(rows_claim(P, P.exec, region, nc), q, pw, qr0.y >> 16, qr0.z);
                        nr++;
                        pw = (pw & ~((7u << 9) | (3u << QP_PEND_SHIFT))) | ((((pw >> 9) & 7u) + 1u) << 9) | (nc << QP_PEND_SHIFT);
                        qtab[q].x = pw;
                    } else {
                        qtab[q].x = pw;
                        if (ready) atomicOr(&qready[(q >> 5) * 32u], 1u << (q & 31u));    // dispatched by the next im_rollout
                    }
                    // the next completion may belong to the same query: its plan word was fetched before this update
                    if (gs1 != ~0u && (cd1.z >> 2) == q) qr1.x = pw;
                    gs0 = gs1; cd0 = cd1; qr0 = qr1; gs1 = gs2; cd1 = cd2;
                }
            }
            ewma_flush();
            // ---- the buffered log records: one claim per warp
            {
                const uint32_t mine = min(nf, 2u);
                const uint32_t b0 = __ballot_sync(kFull, (mine & 1u) != 0), b1 = __ballot_sync(kFull, (mine & 2u) != 0);
                const uint32_t tot = __popc(b0) + 2u * __popc(b1);
                if (tot) {
                    uint32_t base = 0;
                    if (lane == 0) {
                        base = atomicAdd(&P.qlog.cnt[region * kCntStride], tot);
                        if (base + tot > P.qlog.regcap) atomicOr(P.err_flag, 2u);
                    }
                    base = __shfl_sync(kFull, base, 0) + __popc(b0 & lt_mask) + 2u * __popc(b1 & lt_mask);
                    if (mine > 0) P.qlog.rec[(size_t)region * P.qlog.regcap + (base % P.qlog.regcap)] = f_rec[0];
                    if (mine > 1) P.qlog.rec[(size_t)region * P.qlog.regcap + ((base + 1u) % P.qlog.regcap)] = f_rec[1];
                }
            }
            // ---- the buffered executor rows: one claim per warp (a ready query has 1 .. 3 calls in its next stage)
            {
                uint32_t n0 = 0, n1 = 0, a0;
                if (nr > 0) stage_calls((r_pw[0] >> 2) & 3u, (r_pw[0] >> 6) & 7u, (r_pw[0] >> 9) & 7u, a0, n0);
                if (nr > 1) stage_calls((r_pw[1] >> 2) & 3u, (r_pw[1] >> 6) & 7u, (r_pw[1] >> 9) & 7u, a0, n1);
                uint32_t inc = n0 + n1;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { const uint32_t v = __shfl_up_sync(kFull, inc, o); if (lane >= (uint32_t)o) inc += v; }
                const uint32_t tot = __shfl_sync(kFull, inc, 31);
                if (tot) {
                    uint32_t base = 0;
                    if (lane == 0) base = rows_claim(P, P.exec, region, tot);
                    base = __shfl_sync(kFull, base, 0) + inc - (n0 + n1);
                    if (nr > 0) emit_rows(base, r_q[0], r_pw[0], r_io[0], r_dl[0]);
                    if (nr > 1) emit_rows(base + n0, r_q[1], r_pw[1], r_io[1], r_dl[1]);
                }
            }
        }

        // =============================================================== H preempt (R21): largest (deadline, id) first
        if (P.kv_preempt) {
            uint32_t mover = 0;
#pragma unroll 1
            for (uint32_t k = 0; k < N; k++) if (M_KV(k) > s_kvcap[k]) mover |= 1u << k;
#pragma unroll 1
            while (mover) {
                const uint32_t k = __ffs(mover) - 1u;
                mover &= mover - 1u;
                const uint32_t sb = s_sbase[k], cap = s_kvcap[k];
                uint32_t kv = M_KV(k), npre = 0, olo, ohi;
                occ_window(sb, olo, ohi);
                {   // the window also shows the slots of the models behind k: keep the S_k bits of this one
                    const uint32_t S = s_slots[k];
                    if (S < 32) { olo &= (1u << S) - 1u; ohi = 0; }
                    else if (S < 64) ohi &= (1u << (S - 32)) - 1u;
                }
#pragma unroll 1
                while (kv > cap) {
                    uint32_t best = 0, bsl = 0;
                    uint4 bcd = make_uint4(0, 0, 0, 0);
                    // the records of the model's running slots, EIGHT loads in flight at a time (one load per iteration, with
                    // the running maximum carried through it, is a chain of ~12 DRAM round trips per eviction, and with 32 envs
                    // per warp some lane evicts in most ticks).  The loads are unconditional - a slot that is not there reads
                    // the model's first slot and is ignored - so that nothing waits before all eight are out.
#pragma unroll 1
                    for (uint32_t half = 0; half < 2; half++) {
                        uint32_t ob = half ? ohi : olo;
#pragma unroll 1
                        while (ob) {
                            uint32_t sl[8];
                            uint4 cd[8];
                            bool have[8];
#pragma unroll
                            for (int j = 0; j < 8; j++) {
                                have[j] = ob != 0;
                                sl[j] = have[j] ? half * 32u + (uint32_t)__ffs(ob) - 1u : 0u;
                                ob &= ob - 1u;                                              // 0 stays 0
                                cd[j] = cold[2u * (sb + sl[j])];
                            }
#pragma unroll
                            for (int j = 0; j < 8; j++) {
                                const uint32_t key = have[j] ? (((cd[j].x >> 16) << 12) | cd[j].z) + 1u : 0u;   // (deadline, id) + 1; unique
                                if (key > best) { best = key; bsl = sl[j]; bcd = cd[j]; }
                            }
                        }
                    }
                    if (best == 0) break;
                    const uint32_t gs = sb + bsl;
                    uint16_t *hp = hot16 + (gs >> 3) * 256u + (gs & 7u);
                    const uint32_t rem = *hp;
                    *hp = 0;                                                            // a free slot holds 0
                    const uint32_t tm = P.sched_mode ? (bcd.x >> 16) : (bcd.x & 0xFFFFu);
                    list_insert(k, (k << 28) | (tm << 12) | bcd.z, make_uint2((bcd.x & 0xFFFFu) | (rem << 16), bcd.y));   // keeps progress and issue tick; n_wait++
                    if (bsl < 32) olo &= ~(1u << bsl); else ohi &= ~(1u << (bsl - 32));
                    OCC(gs >> 5) &= ~(1u << (gs & 31u));
                    kv -= ((bcd.y >> SW_IN_SHIFT) & SW_TOK_MASK) + ((bcd.y & SW_TOK_MASK) - rem);
                    npre++;
                }
                M_KV(k) = kv;
                M_W0(k) -= npre << 16;                                                   // n_run -= npre
                c_preempt += npre;
            }
        }

        // =============================================================== I record (R27, R28, R33)
        {
            const uint32_t miss_acc = miss + drops_in;
            const unsigned long long cost_acc = cost + ((unsigned long long)drops_in << 16);
            if (active) {
                const size_t idx = (size_t)trow_post * P.E + e;
                P.rew[idx] = __uint2float_rn(rew);
                P.cost[idx] = P.cost_mode ? __uint2float_rn(miss_acc) : __ull2float_rn(cost_acc) * 0x1p-16f;
                P.miss[idx] = (uint8_t)min(miss_acc, 255u);
                P.done[idx] = (uint8_t)done;
            }
#pragma unroll 1
            for (uint32_t k = 0; k < N; k++) { const uint32_t w0 = M_W0(k); c_run += w0 >> 16; c_wait += w0 & 0xFFFFu; }
            if (done) {
                // hard reset: live queries abandoned, pools emptied
                uint32_t live = 0;
#pragma unroll 1
                for (uint32_t w = 0; w < QW; w++) { live += __popc(~QFREE(w)); QFREE(w) = active ? 0xFFFFFFFFu : 0u; qready[w * 32u] = 0; }
                if (active) c_aband += live;
#pragma unroll 1
                for (uint32_t w = 0; w < P.hw_qfree; w++) H(w) = 0;                        // m and occ
#pragma unroll 1
                for (uint32_t g = 0; g < P.n_grp; g++) hot4[g * 32u] = make_uint4(0, 0, 0, 0);
                // the waiting lists: every chunk back on the free list (0 -> 1 -> ... -> end), every model's list empty
#pragma unroll 1
                for (uint32_t w = 0; w < (P.n_chunks + 3u) / 4u; w++) {
                    uint32_t v = 0;
#pragma unroll
                    for (uint32_t jj = 0; jj < 4; jj++) v |= (4u * w + jj + 1u < P.n_chunks ? 4u * w + jj + 1u : 0xFFu) << (8u * jj);
                    H(P.hw_next + w) = v;
                }
#pragma unroll 1
                for (uint32_t w = 0; w < 4; w++) H(P.hw_head + w) = 0xFFFFFFFFu;
                free_head = 0;
            }
        }
    } else {
        bulk::mbar_wait(&s_bar[wib], 0);
        free_head = H(P.hw_misc) >> 16;
    }

    // ===================================================================== pre(t_pre): A arrive, B snapshot, work lists
    uint32_t drops_out = 0;
    if (pre_mode == 1) {
        const int32_t t = t_pre;
        const uint32_t t_rel = (uint32_t)(t - t0);
        // ---- executor rows of queries left ready by an earlier rollout (pending == 0, stages left)
        if (t_post < 0) {
#pragma unroll 1
            for (uint32_t w = 0; w < QW; w++) {
                uint32_t bits = qready[w * 32u];
                if (!__any_sync(kFull, bits != 0)) continue;
                qready[w * 32u] = 0;
#pragma unroll 1
                while (__any_sync(kFull, bits != 0)) {
                    uint32_t q = 0, nc = 0, a0 = 0, pw = 0;
                    uint4 qr = make_uint4(0, 0, 0, 0);
                    const bool have = bits != 0;
                    if (have) {
                        q = w * 32u + (uint32_t)__ffs(bits) - 1u;
                        bits &= bits - 1u;
                        qr = qtab[q];
                        pw = qr.x;
                        stage_calls((pw >> 2) & 3u, (pw >> 6) & 7u, (pw >> 9) & 7u, a0, nc);
                    }
                    uint32_t idx0 = 0;
                    if (claim_exec_rows(nc, idx0) && have) {
                        write_exec_rows(P, region, idx0, e, q, pw, qr.y >> 16, (int32_t)qr.z, t_rel, a0, nc);
                        qtab[q].x = (pw & ~((7u << 9) | (3u << QP_PEND_SHIFT))) | ((((pw >> 9) & 7u) + 1u) << 9) | (nc << QP_PEND_SHIFT);
                    }
                }
            }
        }
        // ---- A arrive (R5, R7, R8, R9)
        {
            const uint32_t n = n_arr_pre;                                // drawn at the top of the kernel
            // the j-th arrival takes the j-th lowest free query index; a full table drops the rest (R9)
            uint32_t nfree = 0;
#pragma unroll 1
            for (uint32_t w = 0; w < QW; w++) nfree += __popc(QFREE(w));
            const uint32_t n_ok = min(n, nfree);
            // planner rows: one claim per warp, lane l writes its rows behind those of the lanes below it
            uint32_t inc = n_ok;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const uint32_t v = __shfl_up_sync(kFull, inc, o); if (lane >= (uint32_t)o) inc += v; }
            const uint32_t ptot = __shfl_sync(kFull, inc, 31);
            uint32_t pbase = 0;
            if (ptot) {
                if (lane == 0) pbase = rows_claim(P, P.plan, region, ptot);
                pbase = __shfl_sync(kFull, pbase, 0) + inc - n_ok;
            }
            uint32_t wq = 0;
#pragma unroll 1
            for (uint32_t j = 0; j < n_ok; j++) {
                while (QFREE(wq) == 0) wq++;
                const uint32_t fb = QFREE(wq), q = wq * 32u + (uint32_t)__ffs(fb) - 1u;
                QFREE(wq) = fb & (fb - 1u);
                const Ph4 d = draw(P, STREAM_QRY, gid, t, j, 0);
                const uint32_t comp = d.z < P.mix_thresh ? 0u : 1u;
                const uint32_t budget = P.mix_lo[comp] + __umulhi(d.x, P.mix_hi[comp] - P.mix_lo[comp] + 1u);
                const uint32_t in_tok = P.has_intok ? __ldg(&P.tab_intok[d.y >> 22]) : P.in_tok_const;
                const int32_t dl = t + (int32_t)budget;                  // PAPER.md:117 deadline = t_arrive + beta
                qtab[q] = make_uint4(QP_LIVE, budget | (in_tok << 16), (uint32_t)dl, (uint32_t)t);
                P.plan.row[region * P.plan.regcap + (pbase + j) % P.plan.regcap] = make_uint4(e, q | (t_rel << 19), (uint32_t)dl, in_tok);
            }
            c_arr += n; c_drop += n - n_ok; c_plans += n_ok;
            drops_out = n - n_ok;                                        // carried to phase I of this tick
            if (active) c_live += P.QCAP - (nfree - n_ok);
        }
    }
    // ---- B snapshot (R14): telemetry features of the state left by the tick just finished.  The policy kernels want
    // the 3N features of an env contiguous; the header sits in shared memory as [word][env], so any lane can read any
    // env's words: lane l takes feature (l & 7) of envs (l >> 3), (l >> 3) + 4, ... and eight lanes write one whole
    // 32-byte sector.  (The eight words of an env are in one bank: an 8-way conflict on 48 loads per block, nothing
    // against the staging pass it replaces.)
    if (pre_mode != 0) {
        const uint32_t *hb = reinterpret_cast<const uint32_t *>(sm);           // word w of env x at hb[w * 32 + x]
        float *snb = P.snap + (size_t)blk * 32u * 3u * N;                      // the block's rows: 32 x 3N contiguous floats
        const uint32_t N3 = 3u * N, n_valid = min(32u, P.E - blk * 32u);
        const uint32_t j = lane & 7u, env0 = lane >> 3;
        __syncwarp();
#pragma unroll 1
        for (uint32_t f = j; f < N3; f += 8) {
            uint32_t word, mask = ~0u;
            float scale;
            if (f < N) { word = 3u * f; mask = 0xFFFFu; scale = 0x1p-6f; }                   // d_queue = n_wait 2^-6
            else if (f < 2u * N) { word = 3u * (f - N) + 2u; scale = 0x1p-18f; }             // d_e2e = ewma_q8 2^-18
            else { word = 3u * (f - 2u * N) + 1u; scale = s_kvinv[f - 2u * N]; }             // d_kv = kv_used * fp32(1 / KV)
            const uint32_t *src = hb + word * 32u + env0;
            float *dst = snb + env0 * N3 + f;
#pragma unroll
            for (uint32_t i = 0; i < 8; i++)
                if (env0 + 4u * i < n_valid) dst[4u * i * N3] = __fmul_rn(__uint2float_rn(src[4u * i] & mask), scale);
        }
    }
    // ---- counters
    {
        const uint32_t cv[C_N] = {c_arr, c_drop, c_fin, c_solved, c_missed, c_issued, c_done, c_preempt, c_soj, c_live, c_plans,
                                  c_issued, c_run, c_wait, 0u, c_aband};
#pragma unroll
        for (int c = 0; c < (int)C_N; c++)
            if (cv[c] != 0) atomicAdd(&ctr[c * 32], cv[c]);      // no return value: a fire-and-forget reduction, no round trip
    }
    // ---- header back to HBM: one bulk copy
    H(P.hw_misc) = drops_out | (free_head << 16);
    H(P.hw_misc + 1u) = 0;
    bulk::fence_proxy_async();
    __syncwarp();
    if (lane == 0) {
        bulk::s2g(blkp, sm, L.hdr_bytes);
        bulk::commit();
        bulk::wait_read();
    }
#undef H
#undef M_W0
#undef M_KV
#undef M_EWMA
#undef OCC
#undef QFREE
#undef NEXTW
#undef HEADW
}

// opt-in to the dynamic shared memory the kernel needs on the CURRENT device (attributes are per device: im_bind calls this)
int sim_prepare_device()
{
    // the kernel lives on shared memory (the resident warps are what hides its latency): ask for the largest carve-out
    if (cudaFuncSetAttribute(k_sim, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared) != cudaSuccess) return -1;
    return cudaFuncSetAttribute(k_sim, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) == cudaSuccess ? 0 : -1;
}

void launch_serve(const Params &P, int32_t t, cudaStream_t st)
{
    const uint32_t warps = P.NB * P.N;
    launch_chained(k_serve, dim3((warps + kServeWarps - 1) / kServeWarps), dim3(kServeWarps * 32), 0, st, true, P, t);
}

void launch_sim(const Params &P, int32_t t_post, uint32_t trow_post, int32_t t_pre, uint32_t pre_mode, int32_t t0, cudaStream_t st)
{
    const SimSmem L = sim_smem(P);
    const uint32_t blocks = (P.NB + kSimWarps - 1) / kSimWarps;
    // the first launch of a rollout (t_post < 0) follows host copies and other kernels: a plain launch
    launch_chained(k_sim, dim3(blocks), dim3(kSimWarps * 32), (size_t)kSimWarps * L.per_warp, st, t_post >= 0, P, L, t_post, trow_post, t_pre, pre_mode, t0);
}

}  // namespace im
