// im_noalloc.cu - im_gae_static (include/inframind.h): the returns kernel for callers that may not allocate.
//
// The GAE / Lagrangian-reward walk of im_returns.cu (Eq. 3; R29, R31: the same sequence of separately
// rounded fp32 operations, so ADV / RET equal those of im_returns bit for bit) as an entry point of its own that takes
// plain device pointers and allocates NOTHING: its scratch memory - the per-CTA partial sums of the cost and the
// ticket that elects the CTA which adds them up - lives in a file-scope `static __device__` array of a fixed, modest
// size that every GPU which loads the library holds until the process exits.
//
// Differences from k_gae: the sum of the cost (the numerator of C-bar, Eq. 7) is not accumulated by
// atomics into memory the caller's ctx owns but written per CTA into the static scratch and added up, in CTA order,
// by the last CTA to finish: no zero-initialised accumulator is needed and the sum is the same in every run.
//
// The array's name is a host-side stand-in in host code, not a device address: the address a kernel can use comes
// from cudaGetSymbolAddress, asked once per device with that device current (scratch_of_current_device).
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/inframind.h"
#include "im_device.cuh"

namespace im {

constexpr int kGsThreads = 256;             // envs per CTA: one thread per env, like k_gae
constexpr int kGsBatch = 16;                // ticks of loads in flight per thread
constexpr uint32_t kGsMaxCtas = IM_GAE_STATIC_MAX_ENVS / kGsThreads;        // 4096
constexpr uint32_t kGsHdrWords = 32;        // 256 bytes: word 0 = ticket, the rest unused (keeps the partials 256-byte aligned)

// scratch: [0] ticket of finished CTAs | [kGsHdrWords + b] cost sum of CTA b (bits of a double)      33 024 bytes
static __device__ __align__(256) unsigned long long g_gae_scratch[kGsHdrWords + kGsMaxCtas];

__global__ void __launch_bounds__(kGsThreads)
k_gae_static(const float *__restrict__ rew, const float *__restrict__ cost, const float *__restrict__ val,
             const uint8_t *__restrict__ done, float *__restrict__ adv, float *__restrict__ ret, uint32_t T, uint32_t E,
             float gamma, float lam, float mu, unsigned long long *__restrict__ scratch, double *__restrict__ sum_cost)
{
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    double csum = 0.0;
    if (e < E) {
        const float gl = __fmul_rn(gamma, lam);
        float A = 0.0f;
        float vnext = val[(size_t)T * E + e];
        int64_t t = (int64_t)T - 1;
        while (t >= 0) {
            const int nb = (int)(t + 1 < kGsBatch ? t + 1 : kGsBatch);
            float r[kGsBatch], c[kGsBatch], v[kGsBatch];
            uint8_t d[kGsBatch];
#pragma unroll
            for (int j = 0; j < kGsBatch; j++)
                if (j < nb) {
                    const size_t i = (size_t)(t - j) * E + e;
                    r[j] = __ldcs(rew + i); c[j] = __ldcs(cost + i); v[j] = __ldcs(val + i); d[j] = __ldcs(done + i);
                }
#pragma unroll
            for (int j = 0; j < kGsBatch; j++)
                if (j < nb) {
                    const size_t i = (size_t)(t - j) * E + e;
                    const bool nd = d[j] == 0;                                                  // R29: no bootstrap across an episode end
                    const float rt = __fsub_rn(r[j], __fmul_rn(mu, c[j]));                      // r - mu C
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
    // cost sum of this CTA -> scratch; the last CTA to arrive adds the partials up in CTA order
#pragma unroll
    for (int o = 16; o; o >>= 1) csum += __shfl_xor_sync(0xffffffffu, csum, o);
    __shared__ double s[kGsThreads / 32];
    __shared__ bool s_last;
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = csum;
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0;
        for (int w = 0; w < kGsThreads / 32; w++) a += s[w];
        scratch[kGsHdrWords + blockIdx.x] = (unsigned long long)__double_as_longlong(a);
        __threadfence();                                                        // the partial is visible before the ticket
        s_last = atomicAdd(&scratch[0], 1ull) == (unsigned long long)gridDim.x - 1ull;
    }
    __syncthreads();
    if (s_last && threadIdx.x < 32) {
        __threadfence();
        double a = 0.0;
        for (uint32_t b = threadIdx.x; b < gridDim.x; b += 32)                  // lane l: CTAs l, l + 32, ... in order
            a += __longlong_as_double((long long)__ldcg(&scratch[kGsHdrWords + b]));
#pragma unroll
        for (int o = 16; o; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
        if (threadIdx.x == 0 && sum_cost) *sum_cost = a;
    }
}

// device address of the scratch array on the CURRENT device: cudaGetSymbolAddress once per device (a module is loaded
// per device, each with its own copy of the array); no allocation
constexpr int kGsMaxDevices = 64;
static std::mutex g_gs_mutex;
static unsigned long long *g_gs_ptr[kGsMaxDevices];

static cudaError_t scratch_of_current_device(unsigned long long **out, int *dev_out)
{
    int dev = -1;
    cudaError_t rc = cudaGetDevice(&dev);
    if (rc != cudaSuccess) return rc;
    *dev_out = dev;
    if (dev < 0 || dev >= kGsMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_gs_mutex);
    if (!g_gs_ptr[dev]) {
        void *p = nullptr;
        rc = cudaGetSymbolAddress(&p, g_gae_scratch);
        if (rc != cudaSuccess) return rc;
        g_gs_ptr[dev] = static_cast<unsigned long long *>(p);
    }
    *out = g_gs_ptr[dev];
    return cudaSuccess;
}

static int gs_fail(char *errbuf, size_t errbuf_bytes, int code, const char *fmt, ...)
{
    if (errbuf && errbuf_bytes) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, errbuf_bytes, fmt, ap);
        va_end(ap);
    }
    return code;
}

}  // namespace im

extern "C" int im_gae_static(const float *rew, const float *cost, const float *val, const uint8_t *done, float *adv, float *ret,
                             double *sum_cost, uint32_t n_ticks, uint32_t n_envs, float gamma, float lambda, float lagrange_mu,
                             void *cuda_stream, char *errbuf, size_t errbuf_bytes)
{
    using namespace im;
    if (errbuf && errbuf_bytes) errbuf[0] = 0;
    if (!rew || !cost || !val || !done || !adv || !ret) return gs_fail(errbuf, errbuf_bytes, IM_ERR_INVALID_ARG, "im_gae_static: null array argument");
    if (n_ticks == 0 || n_envs == 0) return gs_fail(errbuf, errbuf_bytes, IM_ERR_INVALID_ARG, "im_gae_static: n_ticks and n_envs must be positive");
    if (n_envs > IM_GAE_STATIC_MAX_ENVS)
        return gs_fail(errbuf, errbuf_bytes, IM_ERR_CAPACITY,
                       "im_gae_static: n_envs = %u exceeds IM_GAE_STATIC_MAX_ENVS = %u (the static scratch holds one partial sum per 256 envs); "
                       "split the batch by env ranges or use im_returns",
                       n_envs, (unsigned)IM_GAE_STATIC_MAX_ENVS);
    unsigned long long *scratch = nullptr;
    int dev = -1;
    cudaError_t rc = scratch_of_current_device(&scratch, &dev);
    if (rc != cudaSuccess)
        return gs_fail(errbuf, errbuf_bytes, IM_ERR_CUDA, "im_gae_static: scratch address on device %d: %s", dev, cudaGetErrorString(rc));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // the array keeps the previous call's contents: the ticket must start at zero (the partials are all rewritten
    // before they are read)
    rc = cudaMemsetAsync(scratch, 0, kGsHdrWords * sizeof(unsigned long long), st);
    if (rc != cudaSuccess) return gs_fail(errbuf, errbuf_bytes, IM_ERR_CUDA, "im_gae_static: clearing the ticket: %s", cudaGetErrorString(rc));
    const uint32_t ctas = (n_envs + kGsThreads - 1) / kGsThreads;
    k_gae_static<<<ctas, kGsThreads, 0, st>>>(rew, cost, val, done, adv, ret, n_ticks, n_envs, gamma, lambda, lagrange_mu, scratch, sum_cost);
    rc = cudaGetLastError();
    if (rc != cudaSuccess) return gs_fail(errbuf, errbuf_bytes, IM_ERR_CUDA, "im_gae_static: launch: %s", cudaGetErrorString(rc));
    return IM_OK;
}
