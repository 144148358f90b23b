// im_returns.cu — (a) reverse-scan GAE with the Lagrangian reward r - mu*cost (Eq. 3; R29, R31),
// (b) planner utility U_i = solved - mu*L_total/beta and its batch normalisation (Eq. 6; R32),
// (c) the sums behind C-bar of the dual update (Eq. 7).
//
// GAE is a first-order linear recurrence along t for every env independently: one thread per env walks
// t = T-1 .. 0 over [T][E] arrays (E fastest => every load/store of a warp is one coalesced 128-byte line).
// HBM-bound: 13 B read + 8 B written per env-tick.  Loads are issued kBatch ticks ahead of the dependent
// chain so that the walk is bandwidth- not latency-limited.  The arithmetic is the R31 sequence of separately
// rounded fp32 operations.
#include "im_device.cuh"

namespace im {

constexpr int kGaeBatch = 16;           // ticks of loads in flight per thread (13 B each): 8 -> 16 and 128 -> 256 threads per
constexpr int kGaeThreads = 256;        // CTA took the walk from 40 % to the bandwidth of the copy it is measured against

__global__ void __launch_bounds__(kGaeThreads)
k_gae(const float *__restrict__ rew, const float *__restrict__ cost, const float *__restrict__ val,
      const uint8_t *__restrict__ done, float *__restrict__ adv, float *__restrict__ ret, uint32_t T, uint32_t E,
      float gamma, float lam, float mu, double *__restrict__ sums)
{
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    double csum = 0.0;
    if (e < E) {
        const float gl = __fmul_rn(gamma, lam);
        float A = 0.0f;
        float vnext = val[(size_t)T * E + e];
        int64_t t = (int64_t)T - 1;
        while (t >= 0) {
            const int nb = (int)(t + 1 < kGaeBatch ? t + 1 : kGaeBatch);
            float r[kGaeBatch], c[kGaeBatch], v[kGaeBatch];
            uint8_t d[kGaeBatch];
#pragma unroll
            for (int j = 0; j < kGaeBatch; j++)
                if (j < nb) {
                    const size_t i = (size_t)(t - j) * E + e;
                    r[j] = __ldcs(rew + i); c[j] = __ldcs(cost + i); v[j] = __ldcs(val + i); d[j] = __ldcs(done + i);
                }
#pragma unroll
            for (int j = 0; j < kGaeBatch; j++)
                if (j < nb) {
                    const size_t i = (size_t)(t - j) * E + e;
                    const bool nd = d[j] == 0;
                    const float rt = __fsub_rn(r[j], __fmul_rn(mu, c[j]));
                    const float delta = __fsub_rn(__fadd_rn(rt, nd ? __fmul_rn(gamma, vnext) : 0.0f), v[j]);
                    A = __fadd_rn(delta, nd ? __fmul_rn(gl, A) : 0.0f);
                    __stcs(adv + i, A);
                    __stcs(ret + i, __fadd_rn(A, v[j]));
                    vnext = v[j];
                    csum += (double)c[j];
                }
            t -= nb;
        }
    }
    // sum of cost (for C-bar), block reduction then one atomic
#pragma unroll
    for (int o = 16; o; o >>= 1) csum += __shfl_xor_sync(0xffffffffu, csum, o);
    __shared__ double s[kGaeThreads / 32];
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = csum;
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0;
        for (int w = 0; w < kGaeThreads / 32; w++) a += s[w];
        atomicAdd(&sums[0], a);
    }
}

// U_i per finished query; sums[1] += U, sums[2] += U^2, sums[3] += count
__global__ void __launch_bounds__(256)
k_utility(const QLog ql, float mu, double *__restrict__ sums)
{
    const uint32_t region = blockIdx.y;
    const uint32_t n = min(ql.cnt[region * kCntStride], ql.regcap);
    double su = 0.0, su2 = 0.0, cn = 0.0;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const size_t g = (size_t)region * ql.regcap + i;
        const uint4 rec = ql.rec[g];
        const uint32_t info = rec.w;
        const float U = __fsub_rn(__uint2float_rn((info >> 16) & 1u),
                                  __fdiv_rn(__fmul_rn(mu, __uint2float_rn(rec.z)), __uint2float_rn(info & 0xFFFFu)));
        su += (double)U; su2 += (double)U * (double)U; cn += 1.0;
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        su += __shfl_xor_sync(0xffffffffu, su, o); su2 += __shfl_xor_sync(0xffffffffu, su2, o); cn += __shfl_xor_sync(0xffffffffu, cn, o);
    }
    __shared__ double s[3][8];
    if ((threadIdx.x & 31) == 0) { s[0][threadIdx.x >> 5] = su; s[1][threadIdx.x >> 5] = su2; s[2][threadIdx.x >> 5] = cn; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0, b = 0, c = 0;
        for (int w = 0; w < 8; w++) { a += s[0][w]; b += s[1][w]; c += s[2][w]; }
        if (c > 0) { atomicAdd(&sums[1], a); atomicAdd(&sums[2], b); atomicAdd(&sums[3], c); }
    }
}

// (U - mean) / (sigma + 1e-8), population sigma, from the four sums {cost, count, sum U, sum U^2}[4..7] (the job-wide
// sums of an env-sharded run, or a copy of the ctx's own).  U is recomputed from the record, so the pass can be repeated.
__global__ void __launch_bounds__(256)
k_unorm(const QLog ql, float mu, const double *__restrict__ sums)
{
    const uint32_t region = blockIdx.y;
    const uint32_t n = min(ql.cnt[region * kCntStride], ql.regcap);
    const double cnt = sums[3];
    const double mean = cnt > 0 ? sums[1] / cnt : 0.0;
    double var = cnt > 0 ? sums[2] / cnt - mean * mean : 0.0;
    var = var > 0 ? var : 0.0;
    const float fm = (float)mean, fs = (float)(sqrt(var) + 1e-8);
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const size_t g = (size_t)region * ql.regcap + i;
        const uint4 rec = ql.rec[g];
        const float U = __fsub_rn(__uint2float_rn((rec.w >> 16) & 1u),
                                  __fdiv_rn(__fmul_rn(mu, __uint2float_rn(rec.z)), __uint2float_rn(rec.w & 0xFFFFu)));
        ql.unorm[g] = __fdiv_rn(__fsub_rn(U, fm), fs);
    }
}

// sums[4..7] = the sums the normalisation uses: the ctx's own until im_returns_finish supplies the job's
__global__ void k_copy_sums(double *sums) { if (threadIdx.x < 4) sums[4 + threadIdx.x] = sums[threadIdx.x]; }

int launch_unorm(const Params &P, float mu, const double *sums_used, cudaStream_t st)
{
    k_unorm<<<dim3(32, kRegions), 256, 0, st>>>(P.qlog, mu, sums_used);
    return 1;
}

int launch_returns(const Params &P, uint32_t T, float gamma, float lam, float mu, float *adv, float *ret, double *sums, cudaStream_t st)
{
    cudaMemsetAsync(sums, 0, 4 * sizeof(double), st);
    k_gae<<<(P.E + kGaeThreads - 1) / kGaeThreads, kGaeThreads, 0, st>>>(P.rew, P.cost, P.val, P.done, adv, ret, T, P.E, gamma, lam, mu, sums);
    const dim3 grid(32, kRegions);
    k_utility<<<grid, 256, 0, st>>>(P.qlog, mu, sums);
    k_copy_sums<<<1, 32, 0, st>>>(sums);
    k_unorm<<<grid, 256, 0, st>>>(P.qlog, mu, sums + 4);
    return 4;
}

// ------------------------------------------------------------------------------------------------------------------
// Slack-ordered queue (R20): per env, the waiting list sorted with a warp-level bitonic sort — shared-memory staging,
// strides >= 32 exchanged through shared memory, strides < 32 by warp shuffles.  The list key is
// model<<28 | time<<12 | id (im_device.cuh), so ONE u32 sort yields every model's queue in slack order, segment after
// segment.  Serves IM_TEL_QUEUE_ORDER; the admission phase of k_sim extracts only the few smallest keys it can admit.
// ------------------------------------------------------------------------------------------------------------------
constexpr int kQoWarps = 4;

__global__ void __launch_bounds__(kQoWarps * 32)
k_queue_order(const Params P, int32_t t, uint32_t *__restrict__ out)
{
    extern __shared__ __align__(16) uint32_t s_keys[];
    const uint32_t lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const uint32_t e = blockIdx.x * kQoWarps + wib;
    if (e >= P.E) return;
    const uint32_t n_ent = P.n_chunks * kChunk;
    uint32_t n2cap = 32;
    while (n2cap < n_ent) n2cap <<= 1;
    uint32_t *keys = s_keys + (size_t)wib * n2cap;
    // the waiting lists of env e (im_device.cuh): lane k walks the chunks of model k and notes how many entries of each
    // are valid (only the head chunk is partly filled); everything else sorts last as 0xFFFFFFFF
    const uint32_t *wkey = reinterpret_cast<const uint32_t *>(blk_rec(P, e) + P.off_wkey + (size_t)(e & 31u) * P.wkey_stride);
    uint32_t *cnt = s_keys + (size_t)kQoWarps * n2cap + (size_t)wib * P.n_chunks;
    for (uint32_t c = lane; c < P.n_chunks; c += 32) cnt[c] = 0;
    __syncwarp();
    uint32_t n = 0;
    for (uint32_t k = 0; k < P.N; k++) n += *hdr_word(P, e, 3u * k) & 0xFFFFu;
    n = min(n, P.RCAP);
    if (lane < P.N) {
        const uint32_t nk = *hdr_word(P, e, 3u * lane) & 0xFFFFu;
        uint32_t ch = (*hdr_word(P, e, P.hw_head + (lane >> 2)) >> (8u * (lane & 3u))) & 0xFFu, c1 = ((nk - 1u) & (kChunk - 1u)) + 1u;
        for (uint32_t left = nk; left > 0 && ch != 0xFFu; left -= c1, c1 = kChunk) {
            cnt[ch] = c1;
            ch = (*hdr_word(P, e, P.hw_next + (ch >> 2)) >> (8u * (ch & 3u))) & 0xFFu;
        }
    }
    __syncwarp();
    const uint32_t n2 = n2cap;
    for (uint32_t i = lane; i < n2; i += 32)
        keys[i] = (i < n_ent && (i % kChunk) < cnt[i / kChunk]) ? wkey[i] : 0xFFFFFFFFu;
    __syncwarp();
    for (uint32_t k = 2; k <= n2; k <<= 1) {
        uint32_t j = k >> 1;
        for (; j >= 32; j >>= 1) {                 // shared-memory exchanges
            for (uint32_t i = lane; i < n2; i += 32) {
                const uint32_t p = i ^ j;
                if (p > i) {
                    const uint32_t a = keys[i], b = keys[p];
                    const bool up = (i & k) == 0;
                    if ((a > b) == up) { keys[i] = b; keys[p] = a; }
                }
            }
            __syncwarp();
        }
        for (uint32_t it = 0; it < n2; it += 32) { // warp-shuffle exchanges within 32 consecutive keys
            const uint32_t i = it + lane;
            uint32_t v = keys[i];
            const bool up = (i & k) == 0;
            for (uint32_t jj = j; jj > 0; jj >>= 1) {
                const uint32_t o = __shfl_xor_sync(0xffffffffu, v, jj);
                const bool lower = (lane & jj) == 0;
                v = (lower == up) ? (v < o ? v : o) : (v > o ? v : o);
            }
            keys[i] = v;
        }
        __syncwarp();
    }
    uint32_t *o = out + (size_t)e * (P.N + 1 + P.RCAP);
    const uint32_t per_model = lane < P.N ? (*hdr_word(P, e, 3u * lane) & 0xFFFFu) : 0u;    // n_wait of model `lane`
    const uint32_t inc = [&] { uint32_t v = per_model; for (int s = 1; s < 32; s <<= 1) { const uint32_t u = __shfl_up_sync(0xffffffffu, v, s); if (lane >= (uint32_t)s) v += u; } return v; }();
    if (lane < P.N) o[lane + 1] = inc;
    if (lane == 0) o[0] = 0;
    for (uint32_t i = lane; i < P.RCAP; i += 32) o[P.N + 1 + i] = i < n ? (keys[i] & 0xFFFu) : 0xFFFFFFFFu;
}

int launch_queue_order(const Params &P, int32_t t, uint32_t *out, cudaStream_t st)
{
    uint32_t n2cap = 32;
    while (n2cap < P.n_chunks * kChunk) n2cap <<= 1;
    const size_t smem = (size_t)kQoWarps * (n2cap + P.n_chunks) * 4;
    cudaFuncSetAttribute(k_queue_order, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    k_queue_order<<<(P.E + kQoWarps - 1) / kQoWarps, kQoWarps * 32, smem, st>>>(P, t, out);
    return 1;
}

}  // namespace im
