// im_probe.cu - libimprobe.so (include/im_probe.h): the rate at which the device serves accesses at data-dependent
// addresses.  Measurement only; nothing of the method is in here.
#include <cstdint>
#include <cuda_runtime.h>
#include "../../include/im_probe.h"

namespace {

__device__ __forceinline__ uint64_t mix64(uint64_t x)
{
    x ^= x >> 33; x *= 0xff51afd7ed558ccdULL; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ULL; x ^= x >> 33;
    return x;
}
__device__ __forceinline__ void st256(void *p, uint32_t a, uint32_t b)
{
    asm volatile("st.global.v8.b32 [%0], {%1, %2, %1, %2, %1, %2, %1, %2};" ::"l"(p), "r"(a), "r"(b) : "memory");
}

template <int SHAPE>
__global__ void __launch_bounds__(64) k_probe(uint8_t *buf, uint64_t n_windows, uint64_t win_bytes, uint32_t rounds, uint32_t seed, uint32_t *sink)
{
    const uint64_t tid = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x, warp = tid >> 5;
    const uint64_t win_sectors = win_bytes / 32;
    uint32_t acc = 0;
    for (uint32_t it = 0; it < rounds; it++) {
        uint8_t *base = buf + (mix64(warp * 7919ULL + (it >> 3) + seed * 104729ULL) % n_windows) * win_bytes;
        uint8_t *p[4];
#pragma unroll
        for (int i = 0; i < 4; i++) p[i] = base + (mix64(tid * 1315423911ULL + (uint64_t)(it * 4 + i) * 2654435761ULL + seed) % win_sectors) * 32;
        if (SHAPE == IM_PROBE_READ16) {
            uint4 v[4];
#pragma unroll
            for (int i = 0; i < 4; i++) v[i] = *reinterpret_cast<const uint4 *>(p[i]);
#pragma unroll
            for (int i = 0; i < 4; i++) acc += v[i].x ^ v[i].w;
        } else if (SHAPE == IM_PROBE_WRITE16) {
#pragma unroll
            for (int i = 0; i < 4; i++) *reinterpret_cast<uint4 *>(p[i]) = make_uint4(it, i, seed, 0);
        } else if (SHAPE == IM_PROBE_WRITE32) {
#pragma unroll
            for (int i = 0; i < 4; i++) st256(p[i], it, i);
        } else {
            uint32_t v[4];
#pragma unroll
            for (int i = 0; i < 4; i++) v[i] = *reinterpret_cast<const uint32_t *>(p[i]);
#pragma unroll
            for (int i = 0; i < 4; i++) *reinterpret_cast<uint32_t *>(p[i]) = v[i] + 1u;
        }
    }
    if (acc == 0x12345678u) *sink = acc;          // keeps the loads alive
}

}  // namespace

extern "C" int im_probe_random_access(void *dev_buf, size_t bytes, size_t window_bytes, int shape, uint32_t n_threads, uint32_t ops_per_thread,
                                      void *stream, double *gops)
{
    if (!dev_buf || !gops || window_bytes < 4096 || (window_bytes & 31) || bytes < 2 * window_bytes + 64 || shape < 0 || shape >= IM_PROBE_SHAPES ||
        n_threads < 64 || ops_per_thread == 0)
        return -1;
    cudaStream_t st = (cudaStream_t)stream;
    uint8_t *buf = (uint8_t *)dev_buf;
    uint32_t *sink = (uint32_t *)buf;                                   // the first 64 bytes are the probe's own
    buf += 64; bytes -= 64;
    const uint64_t n_windows = bytes / window_bytes;
    const uint32_t blocks = n_threads / 64;
    cudaEvent_t a, b;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return -2;
    for (uint32_t rep = 0; rep < 2; rep++) {
        if (rep == 1) cudaEventRecord(a, st);
        switch (shape) {
        case IM_PROBE_READ16: k_probe<IM_PROBE_READ16><<<blocks, 64, 0, st>>>(buf, n_windows, window_bytes, ops_per_thread, rep, sink); break;
        case IM_PROBE_WRITE16: k_probe<IM_PROBE_WRITE16><<<blocks, 64, 0, st>>>(buf, n_windows, window_bytes, ops_per_thread, rep, sink); break;
        case IM_PROBE_WRITE32: k_probe<IM_PROBE_WRITE32><<<blocks, 64, 0, st>>>(buf, n_windows, window_bytes, ops_per_thread, rep, sink); break;
        default: k_probe<IM_PROBE_RMW4><<<blocks, 64, 0, st>>>(buf, n_windows, window_bytes, ops_per_thread, rep, sink); break;
        }
    }
    cudaEventRecord(b, st);
    float ms = 0.0f;
    const bool ok = cudaEventSynchronize(b) == cudaSuccess && cudaEventElapsedTime(&ms, a, b) == cudaSuccess && cudaGetLastError() == cudaSuccess;
    cudaEventDestroy(a); cudaEventDestroy(b);
    if (!ok || ms <= 0.0f) return -2;
    *gops = (double)blocks * 64.0 * (double)ops_per_thread * 4.0 / ((double)ms * 1e6);
    return 0;
}
