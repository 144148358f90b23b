// im_api.cu — host side of the C ABI declared in include/inframind.h: spec validation, arena carving,
// per-tick launch sequence, telemetry read-back.  No CPU fallback: every compute call needs an sm_100 device.
#include "../../include/inframind.h"
#include "im_device.cuh"
#include <cuda_bf16.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

namespace im {
void launch_sim(const Params &P, int32_t t_post, uint32_t trow_post, int32_t t_pre, uint32_t pre_mode, int32_t t0, cudaStream_t st);
void launch_serve(const Params &P, int32_t t, cudaStream_t st);
int sim_prepare_device();
int policy_prepare_device(const Params &P);
int launch_policy(const Params &P, const Weights &W, bool exec, uint32_t parity, int32_t t0, uint32_t trow, int n_sm, bool bf16, cudaStream_t st);
int launch_returns(const Params &P, uint32_t T, float gamma, float lam, float mu, float *adv, float *ret, double *sums, cudaStream_t st);
int launch_unorm(const Params &P, float mu, const double *sums_used, cudaStream_t st);
int launch_queue_order(const Params &P, int32_t t, uint32_t *out, cudaStream_t st);
size_t f32_smem_bytes(uint32_t F, uint32_t H, uint32_t NOP);
bool tc_supported(uint32_t F, uint32_t H);
size_t tc_image_bytes(bool exec);
void launch_pack_tc(const Weights &W, bool exec, uint32_t n_models, uint32_t f_in, uint32_t hidden, cudaStream_t st);

// empty pools: per 32-env block, zero the SoA-32 parts (header, counters, slot groups: a free slot holds 0, issue list,
// ready bitmap), query bitmap all free for the envs that exist (the padding lanes of the last block have no free slot
// and therefore never admit a query)
__global__ void k_reset(const Params P)
{
    const uint32_t words = P.off_iss / 4;                        // hdr | cm | kvt | ctr | hot
    const size_t n = (size_t)P.NB * words;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const uint32_t b = (uint32_t)(i / words), w = (uint32_t)(i % words), hw = w >> 5;
        uint32_t v = 0;
        if (hw >= P.hw_qfree && hw < P.hw_qfree + P.QW && b * 32u + (w & 31u) < P.E) v = 0xFFFFFFFFu;
        if (hw >= P.hw_head && hw < P.hw_head + 4) v = 0xFFFFFFFFu;                       // every model's list is empty
        if (hw >= P.hw_next && hw < P.hw_head) {                                          // all chunks on the free list: 0 -> 1 -> ... -> end
            const uint32_t c0 = (hw - P.hw_next) * 4u;
            for (uint32_t j = 0; j < 4; j++) v |= (c0 + j + 1u < P.n_chunks ? c0 + j + 1u : 0xFFu) << (8u * j);
        }
        reinterpret_cast<uint32_t *>(P.env_base + (size_t)b * P.blk_stride)[w] = v;
    }
    const uint32_t qw = P.QW * 32u;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < (size_t)P.NB * qw; i += (size_t)gridDim.x * blockDim.x)
        reinterpret_cast<uint32_t *>(P.env_base + (size_t)(i / qw) * P.blk_stride + P.off_qready)[i % qw] = 0;
}

// de-interleave `nw` header / counter words starting at unit `w0` of part `off` into dst[e][nw] (telemetry read-back)
__global__ void k_gather_words(const Params P, uint32_t off, uint32_t w0, uint32_t nw, uint32_t *__restrict__ dst)
{
    const size_t n = (size_t)P.E * nw;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const uint32_t e = (uint32_t)(i / nw), w = (uint32_t)(i % nw);
        dst[i] = reinterpret_cast<const uint32_t *>(P.env_base + (size_t)(e >> 5) * P.blk_stride + off)[(w0 + w) * 32u + (e & 31u)];
    }
}

// a DEVICE blob cannot be checked on the host without a synchronisation: its header is checked here and a mismatch
// raises bit 16 of the error flag (IM_ERR_BAD_SPEC at the next im_read_telemetry)
__global__ void k_check_blob(const uint32_t *h, uint32_t dtype, uint32_t F, uint32_t H, uint32_t n_exec_out, uint32_t *err_flag)
{
    if (threadIdx.x == 0 && (h[0] != 0x494D5042u || h[1] != dtype || h[2] != F || h[3] != H || h[4] != 24u || h[5] != n_exec_out))
        atomicOr(err_flag, 16u);
}

// repack the R26 blob (device copy) into the kernels' layouts
__global__ void k_repack(const uint8_t *blob, uint32_t dtype, uint32_t F, uint32_t H, uint32_t n_out, uint32_t n_out_pad,
                         size_t off_W1, size_t off_b1, size_t off_W2, size_t off_b2, size_t off_W3, size_t off_b3,
                         float *W1t, float *W2t, float *W3t, __nv_bfloat16 *W1, __nv_bfloat16 *W2, __nv_bfloat16 *W3,
                         float *b1, float *b2, float *b3)
{
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
    if (dtype == 0) {
        const float *s1 = (const float *)(blob + off_W1), *s2 = (const float *)(blob + off_W2), *s3 = (const float *)(blob + off_W3);
        for (uint32_t i = tid; i < F * H; i += nth) { const uint32_t o = i / F, k = i % F; W1t[k * H + o] = s1[i]; }
        for (uint32_t i = tid; i < H * H; i += nth) { const uint32_t o = i / H, k = i % H; W2t[k * H + o] = s2[i]; }
        for (uint32_t i = tid; i < H * n_out_pad; i += nth) { const uint32_t k = i / n_out_pad, o = i % n_out_pad; W3t[i] = o < n_out ? s3[o * H + k] : 0.0f; }
    } else {
        const __nv_bfloat16 *s1 = (const __nv_bfloat16 *)(blob + off_W1), *s2 = (const __nv_bfloat16 *)(blob + off_W2), *s3 = (const __nv_bfloat16 *)(blob + off_W3);
        for (uint32_t i = tid; i < F * H; i += nth) W1[i] = s1[i];
        for (uint32_t i = tid; i < H * H; i += nth) W2[i] = s2[i];
        for (uint32_t i = tid; i < H * n_out_pad; i += nth) W3[i] = (i / H) < n_out ? s3[i] : __float2bfloat16(0.0f);
    }
    const float *c1 = (const float *)(blob + off_b1), *c2 = (const float *)(blob + off_b2), *c3 = (const float *)(blob + off_b3);
    for (uint32_t i = tid; i < H; i += nth) { b1[i] = c1[i]; b2[i] = c2[i]; }
    for (uint32_t i = tid; i < n_out_pad; i += nth) b3[i] = i < n_out ? c3[i] : 0.0f;
}
}  // namespace im

using namespace im;

static thread_local std::string g_last_error;

struct im_ctx {
    im_pool_spec spec;
    uint32_t E;
    uint64_t seed;
    std::vector<uint32_t> tab_mult, tab_intok, tab_cdf;
    std::vector<uint8_t> env_level;
    bool bound = false;
    uint8_t *arena = nullptr;
    size_t arena_bytes = 0;
    cudaStream_t stream = nullptr;
    Params P;
    Weights Wp, We;
    uint8_t *d_blob = nullptr;
    size_t blob_bytes = 0;
    std::vector<uint8_t> blob_stage;
    float *adv = nullptr, *ret = nullptr;
    double *sums = nullptr;
    uint32_t *qorder = nullptr;
    int32_t tick = 0, last_t0 = 0;
    uint32_t last_T = 0;
    bool have_returns = false;
    float last_mu = 0.0f;
    uint32_t par_exec = 0, par_plan = 0;
    int n_sm = 148;
    uint64_t launches = 0;
    std::string err;
    // state region (for reset)
    size_t state_off = 0, state_bytes = 0;
    // optional per-kernel-class timing with CUDA events on the bound stream (im_set_profiling)
    bool prof = false;
    std::vector<cudaEvent_t> ev;
    std::vector<int> ev_class;
    size_t ev_used = 0;
    double prof_ms[IM_KERNEL_CLASSES] = {0, 0, 0, 0, 0};
    uint64_t prof_n[IM_KERNEL_CLASSES] = {0, 0, 0, 0, 0};
};

static void prof_begin(im_ctx *c, int cls)
{
    if (!c->prof) return;
    if (c->ev_used + 2 > c->ev.size()) {
        const size_t old = c->ev.size();
        c->ev.resize(old + 1024);
        for (size_t i = old; i < c->ev.size(); i++) cudaEventCreate(&c->ev[i]);
    }
    c->ev_class.push_back(cls);
    cudaEventRecord(c->ev[c->ev_used++], c->stream);
}
static void prof_end(im_ctx *c)
{
    if (!c->prof) return;
    cudaEventRecord(c->ev[c->ev_used++], c->stream);
}
static void prof_collect(im_ctx *c)
{
    for (size_t i = 0; i + 1 < c->ev_used; i += 2) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, c->ev[i], c->ev[i + 1]) == cudaSuccess) {
            const int cls = c->ev_class[i / 2];
            c->prof_ms[cls] += ms; c->prof_n[cls]++;
        }
    }
    c->ev_used = 0; c->ev_class.clear();
}

static int fail(im_ctx *c, int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (c) c->err = buf;
    g_last_error = buf;
    return code;
}

static size_t blob_size(const im_pool_spec &s)
{
    auto pad16 = [](size_t n) { return (n + 15) & ~(size_t)15; };
    const size_t F = s.f_in, H = s.hidden, ws = s.policy_dtype ? 2 : 4;
    size_t b = 32;
    for (int net = 0; net < 2; net++) {
        const size_t no = net ? 3 * s.n_models + 1 : 24;
        b += pad16(H * F * ws) + pad16(H * 4) + pad16(H * H * ws) + pad16(H * 4) + pad16(no * H * ws) + pad16(no * 4);
    }
    return b;
}

static int validate(const im_pool_spec *s, uint32_t E)
{
    if (!s || E == 0) return fail(nullptr, IM_ERR_INVALID_ARG, "null spec or zero envs");
    if (s->abi_version != IM_ABI_VERSION) return fail(nullptr, IM_ERR_BAD_SPEC, "abi_version %u != %u", s->abi_version, IM_ABI_VERSION);
    if (s->n_models == 0 || s->n_models > IM_MAX_MODELS) return fail(nullptr, IM_ERR_BAD_SPEC, "n_models %u out of 1..16", s->n_models);
    if (s->qcap == 0 || s->qcap % 32 || s->qcap > 1024) return fail(nullptr, IM_ERR_BAD_SPEC, "qcap must be a multiple of 32 <= 1024");
    if (s->rcap % 128 || s->rcap < 3 * s->qcap || s->rcap > 4096) return fail(nullptr, IM_ERR_BAD_SPEC, "rcap must be a multiple of 128, >= 3*qcap, <= 4096");
    if (s->max_ticks == 0 || s->max_ticks > 8191) return fail(nullptr, IM_ERR_BAD_SPEC, "max_ticks out of 1..8191");
    if (s->sched_mode > 1 || s->kv_preempt > 1 || s->cost_mode > 1 || s->policy_dtype > 1) return fail(nullptr, IM_ERR_BAD_SPEC, "mode flag out of range");
    if (s->n_levels == 0 || s->n_levels > 256 || s->budget_norm_ticks == 0) return fail(nullptr, IM_ERR_BAD_SPEC, "n_levels / budget_norm_ticks");
    if (s->f_in < 3 * s->n_models + 12) return fail(nullptr, IM_ERR_BAD_SPEC, "f_in %u < 3N+12", s->f_in);
    if (s->policy_dtype == IM_DTYPE_BF16) {
        if (!((s->f_in == 64 && s->hidden == 128) || (s->f_in == 128 && s->hidden == 256)))
            return fail(nullptr, IM_ERR_BAD_SPEC, "bf16 policy supports (f_in,hidden) = (64,128) or (128,256)");
    } else {
        if (s->f_in > 128 || s->hidden > 256 || s->hidden < 8) return fail(nullptr, IM_ERR_BAD_SPEC, "fp32 policy: f_in <= 128, 8 <= hidden <= 256");
        if (f32_smem_bytes(s->f_in, s->hidden, 56) > 200 * 1024) return fail(nullptr, IM_ERR_BAD_SPEC, "fp32 policy too large for shared memory");
    }
    if (!s->out_tok_mult_q16 || !s->arr_cdf || !s->env_level) return fail(nullptr, IM_ERR_INVALID_ARG, "null table pointer");
    for (uint32_t k = 0; k < s->n_models; k++) {
        const im_model_spec &m = s->model[k];
        if (m.slots == 0 || m.slots > 64 || m.kv_cap == 0 || m.rate_tok_s == 0 || m.rate_tok_s > 80000)
            return fail(nullptr, IM_ERR_BAD_SPEC, "model %u: slots out of 1..64, zero kv/rate or rate too large", k);
    }
    for (int i = 0; i < 2; i++)
        if (s->mix_lo[i] == 0 || s->mix_hi[i] < s->mix_lo[i] || s->mix_hi[i] > 65535) return fail(nullptr, IM_ERR_BAD_SPEC, "budget component %d out of range", i);
    for (uint32_t l = 0; l < s->n_levels; l++)
        for (int j = 1; j < 31; j++)
            if (s->arr_cdf[l * 32 + j] < s->arr_cdf[l * 32 + j - 1]) return fail(nullptr, IM_ERR_BAD_SPEC, "arr_cdf row %u not monotone", l);
    for (uint32_t e = 0; e < E; e++)
        if (s->env_level[e] >= s->n_levels) return fail(nullptr, IM_ERR_BAD_SPEC, "env_level[%u] out of range", e);
    uint64_t max_out = 1, max_in = s->in_tok_table ? 0 : s->in_tok_const;
    for (int i = 0; i < 1024; i++) {
        for (int d = 0; d < 3; d++) {
            const uint64_t v = ((uint64_t)s->depth_median_tok[d] * s->out_tok_mult_q16[i]) >> 16;
            max_out = v > max_out ? v : max_out;
        }
        if (s->in_tok_table) max_in = s->in_tok_table[i] > max_in ? s->in_tok_table[i] : max_in;
    }
    if (max_out > 8191 || max_in > 8191) return fail(nullptr, IM_ERR_BAD_SPEC, "output / input tokens exceed 8191 (13-bit fields)");
    for (uint32_t k = 0; k < s->n_models; k++)       // R11: prefill is sub-tick
        if ((uint64_t)s->model[k].prefill_us_per_ktok * (max_in + max_out) / 1000u > 50000u)
            return fail(nullptr, IM_ERR_BAD_SPEC, "model %u: prefill of the largest request exceeds one tick", k);
    if (s->sched_mode > 1) return fail(nullptr, IM_ERR_BAD_SPEC, "sched_mode");
    return IM_OK;
}

// ---- arena carving: the same walk sizes the arena (base == nullptr) and binds the pointers
struct Carver {
    uint8_t *base;
    size_t off = 0;
    template <typename T> T *take(size_t n)
    {
        off = (off + 255) & ~(size_t)255;
        T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
        off += n * sizeof(T);
        return p;
    }
};

// Row capacities of the three lists (whole job).  With IM_FLAG_LOG_DECISIONS the executor / planner lists are linear
// logs of one im_rollout and log_cap_* sizes them (0 = a default from max_ticks).  Without it they are rings that only
// hold one tick's work rows: log_cap_exec / log_cap_plan are ignored and the ring gets a fixed per-tick bound (a tick that
// produces more rows than that is flagged, IM_ERR_CAPACITY at the next read).
static void default_caps(const im_pool_spec &s, uint32_t E, uint64_t &ce, uint64_t &cp, uint64_t &cq)
{
    const bool log = s.debug_flags & IM_FLAG_LOG_DECISIONS;
    const uint64_t per_tick_e = (uint64_t)E * 32 + 4096, per_tick_p = (uint64_t)E * 16 + 4096;
    ce = !log ? per_tick_e : (s.log_cap_exec ? s.log_cap_exec : per_tick_e * s.max_ticks / 8);
    cp = !log ? per_tick_p : (s.log_cap_plan ? s.log_cap_plan : per_tick_p * s.max_ticks / 8);
    cq = s.log_cap_query ? s.log_cap_query : per_tick_p * s.max_ticks / 8;
}

// rows of ONE region: the whole-job capacity scaled by the largest share of envs a region can hold (regions are whole
// 32-env blocks, so small jobs are uneven)
static uint32_t region_cap(uint64_t cap, uint32_t E, uint32_t NB, uint32_t n_regions)
{
    const uint64_t blocks = (NB + n_regions - 1) / n_regions;
    uint64_t envs = blocks * 32;
    if (envs > E) envs = E;
    return (uint32_t)((cap * envs + E - 1) / E) + 64u;
}

static size_t carve(im_ctx *c, const im_pool_spec &s, uint32_t E, uint8_t *base)
{
    Carver cv{base};
    Params P;
    memset(&P, 0, sizeof P);
    const uint32_t N = s.n_models, Q = s.qcap, R = s.rcap;
    const size_t T1 = (size_t)s.max_ticks + 1;
    // ---- one record per block of 32 envs (im_device.cuh): SoA-32 parts, then the per-env arrays
    P.QW = Q / 32;
    P.NB = (E + 31u) / 32u;
    P.n_regions = P.NB < kRegions ? P.NB : kRegions;
    P.slot_base[0] = 0;
    for (uint32_t k = 0; k < kMaxModels; k++) P.slot_base[k + 1] = P.slot_base[k] + (k < N ? ((s.model[k].slots + 7u) & ~7u) : 0u);
    P.SP = P.slot_base[N];
    P.n_grp = P.SP / 8; P.cm_words = (P.n_grp + 3u) / 4u;
    P.n_chunks = R / kChunk + N;                               // <= 4096 / 32 + 16 = 144: chunk ids fit a byte
    P.hw_occ = 3 * N; P.hw_qfree = P.hw_occ + (P.SP + 31u) / 32u + 2u; P.hw_next = P.hw_qfree + P.QW; P.hw_head = P.hw_next + (P.n_chunks + 3u) / 4u;
    P.hw_misc = P.hw_head + 4; P.hdr_words = P.hw_misc + 2;
    auto up128 = [](uint32_t x) { return (x + 127u) & ~127u; };
    uint32_t off = P.hdr_words * 128u;
    P.off_cm = off; off += P.cm_words * 128u;                 // directly behind the header: one bulk copy brings both
    P.off_kvt = off; off += N * 128u;
    P.off_ctr = off; off += (uint32_t)C_N * 128u;
    P.off_hot = off; off += P.n_grp * 512u;
    P.off_iss = off; off += kIssueCap * 256u;
    P.off_qready = off; off += P.QW * 128u;
    P.cold_stride = up128(P.SP * 32u); P.wkey_stride = P.n_chunks * kChunk * 4u; P.waux_stride = P.n_chunks * kChunk * 8u; P.q_stride = Q * 16u;
    P.off_cold = off; off += 32u * P.cold_stride;
    P.off_wkey = off; off += 32u * P.wkey_stride;
    P.off_waux = off; off += 32u * P.waux_stride;
    P.off_q = off; off += 32u * P.q_stride;
    P.blk_stride = up128(off);
    P.env_base = cv.take<uint8_t>((size_t)P.NB * P.blk_stride);
    // ---- control block (zeroed by im_reset)
    cv.off = (cv.off + 255) & ~(size_t)255;
    const size_t ctl_off = cv.off;
    P.snap = cv.take<float>((size_t)E * 3 * N);
    P.err_flag = cv.take<uint32_t>(64);
    P.exec.cnt = cv.take<uint32_t>(kRegions * kCntStride); P.exec.base = cv.take<uint32_t>(2 * kRegions);
    P.plan.cnt = cv.take<uint32_t>(kRegions * kCntStride); P.plan.base = cv.take<uint32_t>(2 * kRegions);
    P.qlog.cnt = cv.take<uint32_t>(kRegions * kCntStride);
    double *sums = cv.take<double>(8);
    const size_t ctl_end = cv.off;
    // ---- tables
    P.tab_mult = cv.take<uint32_t>(1024); P.tab_intok = cv.take<uint32_t>(1024);
    P.tab_cdf = cv.take<uint32_t>((size_t)s.n_levels * 32); P.env_level = cv.take<uint8_t>(E);
    // ---- trajectory
    P.rew = cv.take<float>(T1 * E); P.cost = cv.take<float>(T1 * E); P.val = cv.take<float>(T1 * E);
    P.done = cv.take<uint8_t>(T1 * E); P.miss = cv.take<uint8_t>(T1 * E);
    float *adv = cv.take<float>(T1 * E), *ret = cv.take<float>(T1 * E);
    // ---- row lists / logs
    uint64_t ce, cp, cq;
    default_caps(s, E, ce, cp, cq);
    const uint32_t rce = region_cap(ce, E, P.NB, P.n_regions), rcp = region_cap(cp, E, P.NB, P.n_regions), rcq = region_cap(cq, E, P.NB, P.n_regions);
    P.exec.regcap = rce; P.plan.regcap = rcp; P.qlog.regcap = rcq;
    const size_t ne = (size_t)rce * P.n_regions, np = (size_t)rcp * P.n_regions, nq = (size_t)rcq * P.n_regions;
    const bool log = s.debug_flags & IM_FLAG_LOG_DECISIONS;
    P.exec.row = cv.take<uint4>(ne); P.plan.row = cv.take<uint4>(np);
    if (log) { P.exec.logp = cv.take<float>(ne); P.exec.val = cv.take<float>(ne); P.plan.logp = cv.take<float>(np); }
    P.exec.n_out = 3 * N + 1; P.plan.n_out = 24;
    if (s.debug_flags & IM_FLAG_LOG_LOGITS) { P.exec.logits = cv.take<float>(ne * (3 * N + 1)); P.plan.logits = cv.take<float>(np * 24); }
    P.qlog.rec = cv.take<uint4>(nq);
    P.qlog.unorm = cv.take<float>(nq);
    // ---- weights
    const uint32_t F = s.f_in, H = s.hidden;
    Weights W[2];
    for (int net = 0; net < 2; net++) {
        Weights &w = W[net];
        memset(&w, 0, sizeof w);
        w.n_out = net ? 3 * N + 1 : 24; w.n_out_pad = (w.n_out + 7) & ~7u;
        if (s.policy_dtype == IM_DTYPE_F32) {
            w.W1t = cv.take<float>((size_t)F * H); w.W2t = cv.take<float>((size_t)H * H); w.W3t = cv.take<float>((size_t)H * w.n_out_pad);
        } else {
            w.W1 = cv.take<__nv_bfloat16>((size_t)F * H); w.W2 = cv.take<__nv_bfloat16>((size_t)H * H); w.W3 = cv.take<__nv_bfloat16>((size_t)H * w.n_out_pad);
        }
        w.b1 = cv.take<float>(H); w.b2 = cv.take<float>(H); w.b3 = cv.take<float>(w.n_out_pad);
        if (s.policy_dtype == IM_DTYPE_BF16 && tc_supported(F, H)) w.tc_img = cv.take<uint8_t>(tc_image_bytes(net == 1));
    }
    uint8_t *d_blob = cv.take<uint8_t>(blob_size(s));
    uint32_t *qorder = cv.take<uint32_t>((size_t)E * (N + 1 + R));
    const size_t total = (cv.off + 255) & ~(size_t)255;
    if (c && base) {
        P.E = E; P.N = N; P.QCAP = Q; P.RCAP = R;
        P.sched_mode = s.sched_mode; P.kv_preempt = s.kv_preempt; P.cost_mode = s.cost_mode; P.episode_ticks = s.episode_ticks;
        P.budget_norm = s.budget_norm_ticks; P.in_tok_const = s.in_tok_const; P.mix_thresh = s.mix_thresh; P.env_id_base = s.env_id_base;
        for (int i = 0; i < 2; i++) { P.mix_lo[i] = s.mix_lo[i]; P.mix_hi[i] = s.mix_hi[i]; }
        for (int i = 0; i < 3; i++) P.depth_median[i] = s.depth_median_tok[i];
        P.flags = s.debug_flags; P.has_intok = c->tab_intok.empty() ? 0 : 1;
        P.seed_lo = (uint32_t)c->seed; P.seed_hi = (uint32_t)(c->seed >> 32);
        P.f_in = F; P.hidden = H; P.log_mode = log ? 1 : 0;
        for (uint32_t r = 0; r < 10; r++) {      // R2: key = (seed_lo, seed_hi ^ stream), Weyl increments per round
            P.svc_rk[2 * r] = P.seed_lo + r * 0x9E3779B9u;
            P.svc_rk[2 * r + 1] = (P.seed_hi ^ (uint32_t)STREAM_SVC) + r * 0xBB67AE85u;
        }
        for (uint32_t k = 0; k < N; k++) {
            const im_model_spec &m = s.model[k];
            P.model[k] = ModelTab{m.rate_tok_s, m.slots, m.kv_cap, m.prefill_us_per_ktok, {m.succ_thresh[0], m.succ_thresh[1], m.succ_thresh[2]}, m.kv_inv};
        }
        c->P = P; c->Wp = W[0]; c->We = W[1]; c->d_blob = d_blob; c->blob_bytes = blob_size(s);
        c->adv = adv; c->ret = ret; c->sums = sums; c->qorder = qorder;
        c->state_off = ctl_off; c->state_bytes = ctl_end - ctl_off;
    }
    return total;
}

#define CUDA_TRY(c, expr)                                                                                  \
    do {                                                                                                   \
        cudaError_t _e = (expr);                                                                           \
        if (_e != cudaSuccess) return fail(c, IM_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(_e));        \
    } while (0)

static int copy_out(im_ctx *c, const void *src, size_t bytes, void *dst, size_t cap, size_t *written)
{
    if (written) *written = bytes;
    if (!dst) return IM_OK;
    if (cap < bytes) return fail(c, IM_ERR_CAPACITY, "dst too small: %zu < %zu", cap, bytes);
    CUDA_TRY(c, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return IM_OK;
}

// the append counters of the kRegions regions of a list (one 128-byte line apart on the device)
static int read_counts(im_ctx *c, const uint32_t *dev_cnt, uint32_t (&cnt)[kRegions])
{
    std::vector<uint32_t> h(kRegions * kCntStride);
    CUDA_TRY(c, cudaMemcpy(h.data(), dev_cnt, h.size() * 4, cudaMemcpyDeviceToHost));
    for (uint32_t r = 0; r < kRegions; r++) cnt[r] = h[r * kCntStride];
    return IM_OK;
}

template <typename T>
static int fetch(im_ctx *c, std::vector<T> &h, const T *d, size_t n)
{
    h.resize(n);
    if (n) CUDA_TRY(c, cudaMemcpyAsync(h.data(), d, n * sizeof(T), cudaMemcpyDeviceToHost, c->stream));
    return IM_OK;
}

extern "C" {

size_t im_arena_bytes(const im_pool_spec *spec, uint32_t n_envs)
{
    if (validate(spec, n_envs) != IM_OK) return 0;
    return carve(nullptr, *spec, n_envs, nullptr);
}

int im_create(const im_pool_spec *spec, uint32_t n_envs, uint64_t seed, im_ctx **out)
{
    if (!out) return fail(nullptr, IM_ERR_INVALID_ARG, "out is null");
    *out = nullptr;
    const int rc = validate(spec, n_envs);
    if (rc != IM_OK) return rc;
    im_ctx *c = new (std::nothrow) im_ctx();
    if (!c) return fail(nullptr, IM_ERR_NOMEM, "host allocation failed");
    c->spec = *spec;
    c->E = n_envs; c->seed = seed;
    c->tab_mult.assign(spec->out_tok_mult_q16, spec->out_tok_mult_q16 + 1024);
    if (spec->in_tok_table) c->tab_intok.assign(spec->in_tok_table, spec->in_tok_table + 1024);
    c->tab_cdf.assign(spec->arr_cdf, spec->arr_cdf + (size_t)spec->n_levels * 32);
    c->env_level.assign(spec->env_level, spec->env_level + n_envs);
    c->spec.out_tok_mult_q16 = nullptr; c->spec.in_tok_table = nullptr; c->spec.arr_cdf = nullptr; c->spec.env_level = nullptr;
    *out = c;
    return IM_OK;
}

int im_reset(im_ctx *c)
{
    if (!c) return fail(nullptr, IM_ERR_INVALID_ARG, "ctx is null");
    if (!c->bound) return fail(c, IM_ERR_STATE, "im_reset before im_bind");
    CUDA_TRY(c, cudaMemsetAsync(c->arena + c->state_off, 0, c->state_bytes, c->stream));
    k_reset<<<c->n_sm * 8, 256, 0, c->stream>>>(c->P);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    c->tick = 0; c->last_T = 0; c->have_returns = false; c->par_exec = 0; c->par_plan = 0;
    return IM_OK;
}

int im_bind(im_ctx *c, void *dev_arena, size_t bytes, void *cuda_stream)
{
    if (!c || !dev_arena) return fail(c, IM_ERR_INVALID_ARG, "null ctx or arena");
    if ((uintptr_t)dev_arena & 255) return fail(c, IM_ERR_INVALID_ARG, "arena must be 256-byte aligned");
    int dev = 0, major = 0;
    CUDA_TRY(c, cudaGetDevice(&dev));
    CUDA_TRY(c, cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return fail(c, IM_ERR_CUDA, "device compute capability %d.x is not sm_100 (no fallback path)", major);
    CUDA_TRY(c, cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, dev));
    const size_t need = carve(nullptr, c->spec, c->E, nullptr);
    if (bytes < need) return fail(c, IM_ERR_NOMEM, "arena too small: %zu < %zu", bytes, need);
    c->arena = (uint8_t *)dev_arena; c->arena_bytes = bytes; c->stream = (cudaStream_t)cuda_stream;
    carve(c, c->spec, c->E, c->arena);
    // shared-memory opt-ins are per device: set them for the device this ctx is bound on
    if (sim_prepare_device() || policy_prepare_device(c->P)) return fail(c, IM_ERR_CUDA, "cudaFuncSetAttribute failed on device %d", dev);
    CUDA_TRY(c, cudaMemcpyAsync((void *)c->P.tab_mult, c->tab_mult.data(), 4096, cudaMemcpyHostToDevice, c->stream));
    if (!c->tab_intok.empty()) CUDA_TRY(c, cudaMemcpyAsync((void *)c->P.tab_intok, c->tab_intok.data(), 4096, cudaMemcpyHostToDevice, c->stream));
    else CUDA_TRY(c, cudaMemsetAsync((void *)c->P.tab_intok, 0, 4096, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync((void *)c->P.tab_cdf, c->tab_cdf.data(), c->tab_cdf.size() * 4, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync((void *)c->P.env_level, c->env_level.data(), c->E, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    c->bound = true;
    return im_reset(c);
}

static int upload_weights(im_ctx *c, const void *blob)
{
    cudaPointerAttributes at;
    bool on_device = false;
    if (cudaPointerGetAttributes(&at, blob) == cudaSuccess) on_device = (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged);
    else cudaGetLastError();
    if (!on_device) {
        const uint32_t *h = (const uint32_t *)blob;
        if (h[0] != 0x494D5042u || h[1] != c->spec.policy_dtype || h[2] != c->spec.f_in || h[3] != c->spec.hidden || h[4] != 24 ||
            h[5] != 3 * c->spec.n_models + 1)
            return fail(c, IM_ERR_BAD_SPEC, "policy blob header does not match the spec");
    }
    if (on_device) {
        CUDA_TRY(c, cudaMemcpyAsync(c->d_blob, blob, c->blob_bytes, cudaMemcpyDeviceToDevice, c->stream));
        k_check_blob<<<1, 32, 0, c->stream>>>((const uint32_t *)c->d_blob, c->spec.policy_dtype, c->spec.f_in, c->spec.hidden, 3 * c->spec.n_models + 1, c->P.err_flag);
        c->launches++;
    } else {
        // "a host blob is copied before the call returns": a pinned source would make the async copy truly asynchronous,
        // so the bytes go through a buffer the ctx owns (pageable: the runtime stages it before returning)
        c->blob_stage.assign((const uint8_t *)blob, (const uint8_t *)blob + c->blob_bytes);
        CUDA_TRY(c, cudaMemcpyAsync(c->d_blob, c->blob_stage.data(), c->blob_bytes, cudaMemcpyHostToDevice, c->stream));
    }
    auto pad16 = [](size_t n) { return (n + 15) & ~(size_t)15; };
    const size_t F = c->spec.f_in, H = c->spec.hidden, ws = c->spec.policy_dtype ? 2 : 4;
    size_t off = 32;
    for (int net = 0; net < 2; net++) {
        Weights &w = net ? c->We : c->Wp;
        const size_t oW1 = off; off += pad16(H * F * ws);
        const size_t ob1 = off; off += pad16(H * 4);
        const size_t oW2 = off; off += pad16(H * H * ws);
        const size_t ob2 = off; off += pad16(H * 4);
        const size_t oW3 = off; off += pad16((size_t)w.n_out * H * ws);
        const size_t ob3 = off; off += pad16((size_t)w.n_out * 4);
        k_repack<<<64, 256, 0, c->stream>>>(c->d_blob, c->spec.policy_dtype, (uint32_t)F, (uint32_t)H, w.n_out, w.n_out_pad, oW1, ob1, oW2, ob2, oW3, ob3,
                                            (float *)w.W1t, (float *)w.W2t, (float *)w.W3t, (__nv_bfloat16 *)w.W1, (__nv_bfloat16 *)w.W2,
                                            (__nv_bfloat16 *)w.W3, (float *)w.b1, (float *)w.b2, (float *)w.b3);
        c->launches++;
        if (w.tc_img) { launch_pack_tc(w, net == 1, c->spec.n_models, (uint32_t)F, (uint32_t)H, c->stream); c->launches++; }
    }
    CUDA_TRY(c, cudaGetLastError());
    return IM_OK;
}

int im_rollout(im_ctx *c, const void *policy_weights, uint32_t n_ticks)
{
    if (!c || !policy_weights) return fail(c, IM_ERR_INVALID_ARG, "null ctx or weights");
    if (!c->bound) return fail(c, IM_ERR_STATE, "im_rollout before im_bind");
    if (n_ticks == 0 || n_ticks > c->spec.max_ticks) return fail(c, IM_ERR_CAPACITY, "n_ticks %u out of 1..max_ticks=%u", n_ticks, c->spec.max_ticks);
    {   // absolute ticks (issue, deadline) are 16-bit fields of the device state
        const uint32_t hi = c->spec.mix_hi[0] > c->spec.mix_hi[1] ? c->spec.mix_hi[0] : c->spec.mix_hi[1];
        if ((uint64_t)c->tick + n_ticks + hi >= 65536u) return fail(c, IM_ERR_CAPACITY, "tick %d + %u + budget %u reaches 65536: im_reset first", c->tick, n_ticks, hi);
    }
    int rc = upload_weights(c, policy_weights);
    if (rc != IM_OK) return rc;
    cudaStream_t st = c->stream;
    const Params &P = c->P;
    const bool bf16 = c->spec.policy_dtype == IM_DTYPE_BF16;
    if (P.log_mode) {   // logs restart with every rollout
        CUDA_TRY(c, cudaMemsetAsync(P.exec.cnt, 0, sizeof(uint32_t) * kRegions * kCntStride, st));
        CUDA_TRY(c, cudaMemsetAsync(P.exec.base, 0, sizeof(uint32_t) * 2 * kRegions, st));
        CUDA_TRY(c, cudaMemsetAsync(P.plan.cnt, 0, sizeof(uint32_t) * kRegions * kCntStride, st));
        CUDA_TRY(c, cudaMemsetAsync(P.plan.base, 0, sizeof(uint32_t) * 2 * kRegions, st));
    }
    CUDA_TRY(c, cudaMemsetAsync(P.qlog.cnt, 0, sizeof(uint32_t) * kRegions * kCntStride, st));
    const int32_t t0 = c->tick;
    prof_begin(c, IM_KERNEL_SIM);
    launch_sim(P, -1, 0, t0, 1, t0, st);                                   // A, B of the first tick
    prof_end(c);
    c->launches++;
    for (uint32_t i = 0; i < n_ticks; i++) {
        const int32_t t = t0 + (int32_t)i;
        prof_begin(c, IM_KERNEL_PLAN);
        if (launch_policy(P, c->Wp, false, c->par_plan, t0, i, c->n_sm, bf16, st)) return fail(c, IM_ERR_BAD_SPEC, "unsupported policy shape");
        prof_end(c);
        c->par_plan ^= 1;
        prof_begin(c, IM_KERNEL_EXEC);
        launch_policy(P, c->We, true, c->par_exec, t0, i, c->n_sm, bf16, st);   // C, D: decisions of tick t + critic V[t]
        prof_end(c);
        c->par_exec ^= 1;
        const bool last = (i + 1 == n_ticks);
        prof_begin(c, IM_KERNEL_SERVE);
        launch_serve(P, t, st);                                             // F of tick t
        prof_end(c);
        prof_begin(c, IM_KERNEL_SIM);
        launch_sim(P, t, i, t + 1, last ? 2u : 1u, t0, st);                 // D-issue, E, G .. I of tick t, A, B of tick t+1
        prof_end(c);
        c->launches += 4;
    }
    prof_begin(c, IM_KERNEL_EXEC);
    launch_policy(P, c->We, true, c->par_exec, t0, n_ticks, c->n_sm, bf16, st);  // bootstrap V[n_ticks] (R30)
    prof_end(c);
    c->par_exec ^= 1;
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    c->tick = t0 + (int32_t)n_ticks; c->last_t0 = t0; c->last_T = n_ticks; c->have_returns = false;
    return IM_OK;
}

int im_returns(im_ctx *c, float gamma, float lambda, float lagrange_mu)
{
    if (!c) return fail(nullptr, IM_ERR_INVALID_ARG, "ctx is null");
    if (!c->bound || c->last_T == 0) return fail(c, IM_ERR_STATE, "im_returns before im_rollout");
    prof_begin(c, IM_KERNEL_RETURNS);
    c->launches += launch_returns(c->P, c->last_T, gamma, lambda, lagrange_mu, c->adv, c->ret, c->sums, c->stream);
    prof_end(c);
    CUDA_TRY(c, cudaGetLastError());
    c->have_returns = true; c->last_mu = lagrange_mu;
    return IM_OK;
}

int im_returns_finish(im_ctx *c, const double *global_sums)
{
    if (!c || !global_sums) return fail(c, IM_ERR_INVALID_ARG, "null ctx or sums");
    if (!c->bound || !c->have_returns) return fail(c, IM_ERR_STATE, "im_returns_finish before im_returns");
    // device order of the sums: {cost, sum U, sum U^2, count}; the job-wide ones live behind the ctx's own
    const double dev[4] = {global_sums[0], global_sums[2], global_sums[3], global_sums[1]};
    CUDA_TRY(c, cudaMemcpyAsync(c->sums + 4, dev, sizeof dev, cudaMemcpyHostToDevice, c->stream));   // pageable source: staged before the call returns
    prof_begin(c, IM_KERNEL_RETURNS);
    c->launches += launch_unorm(c->P, c->last_mu, c->sums + 4, c->stream);
    prof_end(c);
    CUDA_TRY(c, cudaGetLastError());
    return IM_OK;
}

int im_read_telemetry(im_ctx *c, uint32_t what, void *dst, size_t dst_bytes, size_t *written)
{
    if (!c) return fail(nullptr, IM_ERR_INVALID_ARG, "ctx is null");
    if (!c->bound) return fail(c, IM_ERR_STATE, "im_read_telemetry before im_bind");
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    const Params &P = c->P;
    uint32_t flag = 0;
    CUDA_TRY(c, cudaMemcpy(&flag, P.err_flag, 4, cudaMemcpyDeviceToHost));
    if (flag & 16u) return fail(c, IM_ERR_BAD_SPEC, "device policy blob header does not match the spec");
    if (flag) return fail(c, IM_ERR_CAPACITY, "log / work-list overflow during rollout (flag %u): raise log_cap_*", flag);
    const size_t E = c->E, T = c->last_T, N = P.N, Q = P.QCAP, R = P.RCAP;
    switch (what) {
    case IM_TEL_REW: return copy_out(c, P.rew, 4 * T * E, dst, dst_bytes, written);
    case IM_TEL_COST: return copy_out(c, P.cost, 4 * T * E, dst, dst_bytes, written);
    case IM_TEL_VAL: return copy_out(c, P.val, 4 * (T + 1) * E, dst, dst_bytes, written);
    case IM_TEL_DONE: return copy_out(c, P.done, T * E, dst, dst_bytes, written);
    case IM_TEL_MISS: return copy_out(c, P.miss, T * E, dst, dst_bytes, written);
    case IM_TEL_ADV:
    case IM_TEL_RET:
        if (!c->have_returns) return fail(c, IM_ERR_STATE, "ADV/RET read before im_returns");
        return copy_out(c, what == IM_TEL_ADV ? c->adv : c->ret, 4 * T * E, dst, dst_bytes, written);
    case IM_TEL_COUNTERS:
    case IM_TEL_SNAPSHOT: {
        // the device keeps these struct-of-arrays across the 32 envs of a block: gather them per env, then widen / unpack
        const bool ctr = what == IM_TEL_COUNTERS;
        const size_t nw = ctr ? (size_t)C_N : 3 * N, bytes = ctr ? 128 * E : 16 * N * E;
        if (written) *written = bytes;
        if (!dst) return IM_OK;
        if (dst_bytes < bytes) return fail(c, IM_ERR_CAPACITY, "dst too small: %zu < %zu", dst_bytes, bytes);
        k_gather_words<<<c->n_sm * 4, 256, 0, c->stream>>>(P, ctr ? P.off_ctr : 0u, 0u, (uint32_t)nw, c->qorder);
        c->launches++;
        CUDA_TRY(c, cudaGetLastError());
        std::vector<uint32_t> h;
        int rc = fetch(c, h, c->qorder, E * nw);
        if (rc) return rc;
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
        if (ctr) {
            uint64_t *o = (uint64_t *)dst;
            for (size_t i = 0; i < E * nw; i++) o[i] = h[i];
        } else {
            uint32_t *o = (uint32_t *)dst;
            for (size_t e = 0; e < E; e++)
                for (size_t k = 0; k < N; k++) {
                    const uint32_t *m = &h[e * nw + 3 * k];
                    uint32_t *r = o + (e * N + k) * 4;
                    r[0] = m[0] & 0xFFFFu; r[1] = m[0] >> 16; r[2] = m[1]; r[3] = m[2];
                }
        }
        return IM_OK;
    }
    case IM_TEL_TABLES: {
        const size_t bytes = 4096 + 4096 + c->tab_cdf.size() * 4;
        if (written) *written = bytes;
        if (!dst) return IM_OK;
        if (dst_bytes < bytes) return fail(c, IM_ERR_CAPACITY, "dst too small");
        CUDA_TRY(c, cudaMemcpy(dst, P.tab_mult, 4096, cudaMemcpyDeviceToHost));
        CUDA_TRY(c, cudaMemcpy((uint8_t *)dst + 4096, P.tab_intok, 4096, cudaMemcpyDeviceToHost));
        CUDA_TRY(c, cudaMemcpy((uint8_t *)dst + 8192, P.tab_cdf, c->tab_cdf.size() * 4, cudaMemcpyDeviceToHost));
        return IM_OK;
    }
    case IM_TEL_SCALARS: {
        if (written) *written = 64;
        if (!dst) return IM_OK;
        if (dst_bytes < 64) return fail(c, IM_ERR_CAPACITY, "dst too small");
        double s[8] = {0, 0, 0, 0, 0, 0, 0, 0}, out[8];
        if (c->have_returns) CUDA_TRY(c, cudaMemcpy(s, c->sums + 4, 32, cudaMemcpyDeviceToHost));   // the sums in use: own, or the job's
        uint32_t ce[kRegions], cp[kRegions];
        if (int rc = read_counts(c, P.exec.cnt, ce)) return rc;
        if (int rc = read_counts(c, P.plan.cnt, cp)) return rc;
        double ne = 0, np = 0;
        for (uint32_t r = 0; r < kRegions; r++) { ne += ce[r]; np += cp[r]; }
        const double cnt = s[3], mean = cnt > 0 ? s[1] / cnt : 0.0;
        double var = cnt > 0 ? s[2] / cnt - mean * mean : 0.0;
        var = var > 0 ? var : 0.0;
        out[0] = cnt > 0 ? s[0] / cnt : 0.0; out[1] = mean; out[2] = std::sqrt(var); out[3] = s[0]; out[4] = cnt;
        out[5] = P.log_mode ? ne : -1.0; out[6] = P.log_mode ? np : -1.0; out[7] = (double)c->tick;
        memcpy(dst, out, 64);
        return IM_OK;
    }
    case IM_TEL_SUMS: {
        if (!c->have_returns) return fail(c, IM_ERR_STATE, "SUMS read before im_returns");
        if (written) *written = 32;
        if (!dst) return IM_OK;
        if (dst_bytes < 32) return fail(c, IM_ERR_CAPACITY, "dst too small");
        double s[4];
        CUDA_TRY(c, cudaMemcpy(s, c->sums, 32, cudaMemcpyDeviceToHost));
        const double out[4] = {s[0], s[3], s[1], s[2]};           // sum cost, n finalised, sum U, sum U^2
        memcpy(dst, out, 32);
        return IM_OK;
    }
    case IM_TEL_DECISIONS_EXEC:
    case IM_TEL_DECISIONS_PLAN:
    case IM_TEL_LOGITS_EXEC:
    case IM_TEL_LOGITS_PLAN: {
        if (!P.log_mode) return fail(c, IM_ERR_STATE, "decision log needs IM_FLAG_LOG_DECISIONS");
        const bool ex = what == IM_TEL_DECISIONS_EXEC || what == IM_TEL_LOGITS_EXEC;
        const bool lg = what == IM_TEL_LOGITS_EXEC || what == IM_TEL_LOGITS_PLAN;
        const RowBuf &rb = ex ? P.exec : P.plan;
        if (lg && !rb.logits) return fail(c, IM_ERR_STATE, "logits need IM_FLAG_LOG_LOGITS");
        uint32_t cnt[kRegions];
        if (int rc = read_counts(c, rb.cnt, cnt)) return rc;
        size_t n = 0;
        for (uint32_t r = 0; r < kRegions; r++) n += cnt[r];
        const size_t rec = lg ? 4 * rb.n_out : 24;
        if (written) *written = n * rec;
        if (!dst) return IM_OK;
        if (dst_bytes < n * rec) return fail(c, IM_ERR_CAPACITY, "dst too small: %zu < %zu", dst_bytes, n * rec);
        size_t k = 0;
        for (uint32_t r = 0; r < kRegions; r++) {
            const size_t m = cnt[r], o = (size_t)r * rb.regcap;
            if (!m) continue;
            if (lg) {
                CUDA_TRY(c, cudaMemcpy((uint8_t *)dst + k * rec, rb.logits + o * rb.n_out, m * rec, cudaMemcpyDeviceToHost));
            } else {
                std::vector<uint4> row;
                std::vector<uint32_t> lp, vl;
                int rc;
                if ((rc = fetch(c, row, rb.row + o, m)) || (rc = fetch(c, lp, (const uint32_t *)rb.logp + o, m))) return rc;
                if (ex && (rc = fetch(c, vl, (const uint32_t *)rb.val + o, m))) return rc;
                CUDA_TRY(c, cudaStreamSynchronize(c->stream));
                uint32_t *out = (uint32_t *)dst + k * 6;
                for (size_t i = 0; i < m; i++) {
                    const uint32_t a = row[i].y;
                    out[i * 6 + 0] = P.env_id_base + row[i].x;
                    out[i * 6 + 1] = (uint32_t)(c->last_t0 + (int32_t)(a >> 19));
                    out[i * 6 + 2] = ex ? ((a & 0x3FFu) | (((a >> 10) & 3u) << 16)) : (a & 0x3FFu);
                    out[i * 6 + 3] = row[i].w >> 16;
                    out[i * 6 + 4] = lp[i];
                    out[i * 6 + 5] = ex ? vl[i] : 0u;
                }
            }
            k += m;
        }
        return IM_OK;
    }
    case IM_TEL_QUERIES:
    case IM_TEL_UNORM: {
        if (what == IM_TEL_UNORM && !c->have_returns) return fail(c, IM_ERR_STATE, "UNORM read before im_returns");
        uint32_t cnt[kRegions];
        if (int rc = read_counts(c, P.qlog.cnt, cnt)) return rc;
        size_t n = 0;
        for (uint32_t r = 0; r < kRegions; r++) n += cnt[r];
        const size_t rec = what == IM_TEL_QUERIES ? 16 : 4;
        if (written) *written = n * rec;
        if (!dst) return IM_OK;
        if (dst_bytes < n * rec) return fail(c, IM_ERR_CAPACITY, "dst too small: %zu < %zu", dst_bytes, n * rec);
        size_t k = 0;
        for (uint32_t r = 0; r < kRegions; r++) {
            const size_t m = cnt[r], o = (size_t)r * P.qlog.regcap;
            if (!m) continue;
            if (what == IM_TEL_UNORM) CUDA_TRY(c, cudaMemcpy((float *)dst + k, P.qlog.unorm + o, 4 * m, cudaMemcpyDeviceToHost));
            else CUDA_TRY(c, cudaMemcpy((uint32_t *)dst + k * 4, P.qlog.rec + o, 16 * m, cudaMemcpyDeviceToHost));
            k += m;
        }
        return IM_OK;
    }
    case IM_TEL_STATE: {
        const size_t RD = 4 * Q;                                  // canonical request table: row = 4*query + agent
        const size_t words = 4 * N + 4 * Q + 5 * RD, bytes = 4 * words * E;
        if (written) *written = bytes;
        if (!dst) return IM_OK;
        if (dst_bytes < bytes) return fail(c, IM_ERR_CAPACITY, "dst too small: %zu < %zu", dst_bytes, bytes);
        std::vector<uint8_t> buf;
        const size_t batch = 8;                                   // blocks of 32 envs per copy
        uint32_t *w = (uint32_t *)dst;
        for (size_t b0 = 0; b0 < P.NB; b0 += batch) {
            const size_t nb = P.NB - b0 < batch ? P.NB - b0 : batch;
            buf.resize(nb * P.blk_stride);
            CUDA_TRY(c, cudaMemcpy(buf.data(), P.env_base + b0 * P.blk_stride, nb * P.blk_stride, cudaMemcpyDeviceToHost));
            for (size_t e = b0 * 32; e < (b0 + nb) * 32 && e < E; e++) {
                const uint8_t *blk = buf.data() + (e / 32 - b0) * P.blk_stride;
                const size_t l = e & 31;
                const uint32_t *hdr = (const uint32_t *)blk;
                auto H = [&](uint32_t wd) { return hdr[wd * 32 + l]; };
                const uint16_t *hot = (const uint16_t *)(blk + P.off_hot);
                const uint32_t *wkey = (const uint32_t *)(blk + P.off_wkey + l * P.wkey_stride);
                const uint4 *cold = (const uint4 *)(blk + P.off_cold + l * P.cold_stride), *qt = (const uint4 *)(blk + P.off_q + l * P.q_stride);
                const uint2 *waux = (const uint2 *)(blk + P.off_waux + l * P.waux_stride);
                for (uint32_t k = 0; k < N; k++, w += 4) { w[0] = H(3 * k) & 0xFFFFu; w[1] = H(3 * k) >> 16; w[2] = H(3 * k + 1); w[3] = H(3 * k + 2); }
                for (size_t i = 0; i < Q; i++, w += 4) {
                    if ((H(P.hw_qfree + (uint32_t)(i >> 5)) >> (i & 31)) & 1u) { w[0] = w[1] = w[2] = w[3] = 0; continue; }
                    w[0] = qt[i].x; w[1] = qt[i].z; w[2] = qt[i].w; w[3] = qt[i].y;
                }
                memset(w, 0, 4 * 5 * RD);
                auto put = [&](uint32_t id, uint32_t state, uint32_t model, uint32_t sw, uint32_t dl, uint32_t issue, uint32_t rem, uint32_t slot1) {
                    uint32_t *r = w + 5 * (size_t)id;
                    r[0] = state | (model << 2) | (((sw >> SW_DEPTH_SHIFT) & 3u) << 6) | ((id & 3u) << 8) | (((sw >> SW_SUCC_SHIFT) & 1u) << 10) | ((id >> 2) << 16);
                    r[1] = dl; r[2] = issue; r[3] = rem | (slot1 << 16);
                    r[4] = (sw & SW_TOK_MASK) | (((sw >> SW_IN_SHIFT) & SW_TOK_MASK) << 16);
                };
                for (uint32_t k = 0; k < N; k++)
                    for (uint32_t sl = 0; sl < c->spec.model[k].slots; sl++) {
                        const uint32_t gs = P.slot_base[k] + sl;
                        if (!((H(P.hw_occ + (gs >> 5)) >> (gs & 31)) & 1u)) continue;
                        const uint32_t rem = hot[((gs >> 3) * 32 + l) * 8 + (gs & 7)];
                        put(cold[2 * gs].z & 0xFFFu, ST_RUN, k, cold[2 * gs].y, cold[2 * gs].x >> 16, cold[2 * gs].x & 0xFFFFu, rem, sl + 1);
                    }
                for (uint32_t k = 0; k < N; k++) {                            // waiting lists: model k's chunks, the head chunk partly filled
                    const uint32_t n = H(3 * k) & 0xFFFFu;
                    uint32_t ch = (H(P.hw_head + (k >> 2)) >> (8 * (k & 3))) & 0xFFu, cnt = ((n - 1u) & (kChunk - 1u)) + 1u;
                    for (uint32_t left = n; left > 0 && ch != 0xFFu; left -= cnt, cnt = kChunk) {
                        for (uint32_t j = ch * kChunk; j < ch * kChunk + cnt; j++) {
                            const uint32_t key = wkey[j];
                            const uint32_t id = key & 0xFFFu, tm = (key >> 12) & 0xFFFFu;
                            put(id, ST_WAIT, key >> 28, waux[j].y, P.sched_mode ? tm : qt[id >> 2].z, waux[j].x & 0xFFFFu, waux[j].x >> 16, 0);
                        }
                        ch = (H(P.hw_next + (ch >> 2)) >> (8 * (ch & 3))) & 0xFFu;
                    }
                }
                w += 5 * RD;
            }
        }
        return IM_OK;
    }
    case IM_TEL_QUEUE_ORDER: {
        c->launches += launch_queue_order(P, c->tick, c->qorder, c->stream);
        CUDA_TRY(c, cudaGetLastError());
        return copy_out(c, c->qorder, 4 * E * (N + 1 + R), dst, dst_bytes, written);
    }
    default: return fail(c, IM_ERR_INVALID_ARG, "unknown telemetry selector %u", what);
    }
}

int im_device_ptr(im_ctx *c, uint32_t what, void **dev_ptr, size_t *bytes)
{
    if (!c || !dev_ptr || !bytes) return fail(c, IM_ERR_INVALID_ARG, "null argument");
    if (!c->bound) return fail(c, IM_ERR_STATE, "not bound");
    const size_t E = c->E, T = c->last_T;
    switch (what) {
    case IM_TEL_REW: *dev_ptr = c->P.rew; *bytes = 4 * T * E; break;
    case IM_TEL_COST: *dev_ptr = c->P.cost; *bytes = 4 * T * E; break;
    case IM_TEL_VAL: *dev_ptr = c->P.val; *bytes = 4 * (T + 1) * E; break;
    case IM_TEL_DONE: *dev_ptr = c->P.done; *bytes = T * E; break;
    case IM_TEL_MISS: *dev_ptr = c->P.miss; *bytes = T * E; break;
    case IM_TEL_ADV:
    case IM_TEL_RET:
        if (!c->have_returns) return fail(c, IM_ERR_STATE, "ADV/RET before im_returns");
        *dev_ptr = what == IM_TEL_ADV ? c->adv : c->ret; *bytes = 4 * T * E; break;
    default: return fail(c, IM_ERR_INVALID_ARG, "selector %u has no device array", what);
    }
    return IM_OK;
}

uint64_t im_launch_count(const im_ctx *c) { return c ? c->launches : 0; }

int im_set_profiling(im_ctx *c, int enable)
{
    if (!c) return fail(nullptr, IM_ERR_INVALID_ARG, "ctx is null");
    if (c->bound) { cudaStreamSynchronize(c->stream); prof_collect(c); }
    c->prof = enable != 0;
    return IM_OK;
}

int im_kernel_times(im_ctx *c, double *ms, uint64_t *launches)
{
    if (!c || !ms || !launches) return fail(c, IM_ERR_INVALID_ARG, "null argument");
    if (c->bound) { CUDA_TRY(c, cudaStreamSynchronize(c->stream)); prof_collect(c); }
    for (int i = 0; i < IM_KERNEL_CLASSES; i++) { ms[i] = c->prof_ms[i]; launches[i] = c->prof_n[i]; c->prof_ms[i] = 0; c->prof_n[i] = 0; }
    return IM_OK;
}

void im_destroy(im_ctx *c)
{
    if (!c) return;
    if (c->bound) cudaStreamSynchronize(c->stream);
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    delete c;
}

const char *im_last_error(const im_ctx *c) { return c ? c->err.c_str() : g_last_error.c_str(); }

}  // extern "C"
