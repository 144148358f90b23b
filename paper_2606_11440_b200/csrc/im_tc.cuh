// im_tc.cuh — sm_100a tensor-core building blocks of the bf16 policy path (reading R25):
// inline-PTX wrappers for tcgen05 (TMEM allocation, UMMA issue, TMEM load/store, commit) and mbarrier, the shared
// memory operand layout, and the three-layer MLP of one 128-row tile.
//
// Operand layout ("canonical K-major, no swizzle"): a [rows][K] bf16 matrix is stored as 16-byte chunks of 8
// consecutive k, chunk-major:  byte offset(r, k) = (k / 8) * rows * 16 + r * 16 + (k % 8) * 2.
// A core matrix (8 rows x 16 bytes) is then 128 contiguous bytes; in the UMMA shared-memory descriptor the stride
// between 8-row groups (SBO) is 128 B and the stride between k-chunks (LBO) is rows * 16 B.
//
// Tile data flow: see TcMlp below.  The hidden activations never touch shared memory: all three weight matrices
// stay resident in it instead.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace im {
namespace tc {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---------------------------------------------------------------------------------------------- mbarrier
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n\t"
        ".reg .pred P1;\n\t"
        "LAB_WAIT:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
        "@P1 bra DONE;\n\t"
        "bra LAB_WAIT;\n\t"
        "DONE:\n\t"
        "}" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}

// ---------------------------------------------------------------------------------------------- fences
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tc_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// ---------------------------------------------------------------------------------------------- TMEM
// one full warp allocates `cols` (power of two >= 32) columns; the base address lands in *slot (shared memory)
__device__ __forceinline__ void tmem_alloc(uint32_t *slot, uint32_t cols)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot)), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t base, uint32_t cols)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "r"(cols) : "memory");
}

// ---------------------------------------------------------------------------------------------- descriptors
// shared-memory matrix descriptor, K-major, SWIZZLE_NONE, version 1 (sm_100)
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    return (uint64_t)((saddr >> 4) & 0x3FFFu) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32) | (1ull << 46);
}
// instruction descriptor of kind::f16: D fp32, A and B bf16, both K-major, dense
__host__ __device__ constexpr uint32_t instr_desc_bf16(uint32_t M, uint32_t N)
{
    return (1u << 4) | (1u << 7) | (1u << 10) | ((N >> 3) << 17) | ((M >> 4) << 24);
}

// D[tmem] (+)= A[smem] * B[smem]^T — issued by ONE thread
__device__ __forceinline__ void umma_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem]^T
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t"
        "}" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// One lane of a CONVERGED warp (elect.sync).  UMMAs are issued this way - `if (warp-uniform condition) if (elect_one())` -
// and never under a per-thread condition such as threadIdx.x == 0: there ptxas cannot prove the operands uniform and
// wraps every UTCHMMA in an elect / broadcast / branch loop of ~15 dependent instructions (measured: 62 cycles per
// UMMA, 2000 cycles of blocking issue for layer 2).
__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile(
        "{\n\t"
        ".reg .pred P;\n\t"
        "elect.sync _|P, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, P;\n\t"
        "}" : "=r"(pred));
    return pred != 0;
}
// all UMMAs issued so far by this thread arrive on `bar` when they complete (implies fence::before_thread_sync)
__device__ __forceinline__ void umma_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// ---------------------------------------------------------------------------------------------- TMEM <-> registers
// warp-collective: lane i of the warp reads 32 consecutive columns of TMEM lane (taddr.lane + i)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
          "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
          "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
          "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
          "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ uint32_t tmem_ld1(uint32_t taddr)
{
    uint32_t v;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v) : "r"(taddr) : "memory");
    return v;
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[16])
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
        "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]), "r"(v[10]),
        "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
        : "memory");
}

__device__ __forceinline__ float tanh_approx(float x)
{
    float y;
    asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// (a.x + b.x, a.y + b.y) in one instruction (sm_100 packed fp32 add; each half rounds like a scalar add.rn)
__device__ __forceinline__ float2 fadd2(uint32_t ax, uint32_t ay, float2 b)
{
    unsigned long long ra, rb, rd;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ra) : "r"(ax), "r"(ay));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rb) : "f"(b.x), "f"(b.y));
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
    float2 d;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(rd));
    return d;
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi)
{
    const __nv_bfloat162 p = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<const uint32_t *>(&p);
}

// byte offset of element (r, k) of a [rows][K] bf16 operand in the canonical layout
__host__ __device__ constexpr uint32_t canon_off(uint32_t rows, uint32_t r, uint32_t k) { return (k >> 3) * rows * 16u + r * 16u + (k & 7u) * 2u; }


// ---------------------------------------------------------------------------------------------- the MLP of one tile
// Shared-memory image of one net (built once by k_pack_tc, copied verbatim by every CTA):
//   [ W1 canon [H][K1] | W2 canon [H][H] | W3 canon [NO][H] | b1[H] b2[H] b3[NO] fp32 ]
//
// Two warpgroups (256 threads) share a tile as a two-stage pipeline.  Warpgroup 1 owns layer 1: features into shared
// memory, issue of layer 1, both tanh halves (half a while the tensor core computes half b), issue of layer 2, and -
// behind layer 2 in the tensor pipe - layer 1 of the NEXT tile.  Warpgroup 0 owns layer 2's tanh, layer 3 and the
// sampling epilogue.  So the hidden phases of consecutive tiles overlap.  Everything is packed in place:
//   D1 = [0,256) -> A2 = [0,128) ; D2 = [256,512) -> A3 = [256,320) u [384,448) ; D3 = [448,512)
// and the only cross-tile hazard is layer 2 of tile i+1 (D2) over D3 / A3 of tile i: its issue waits for the logits.
template <int K1, int H, int NO>
struct TcMlp {
    static_assert(K1 % 16 == 0 && H == 256 && NO % 16 == 0 && NO <= 64, "shape");
    static constexpr uint32_t kW1 = 0, kW2 = kW1 + H * K1 * 2, kW3 = kW2 + H * H * 2, kBias = kW3 + NO * H * 2;
    static constexpr uint32_t kImageBytes = kBias + (2 * H + NO) * 4;
    static constexpr uint32_t kA1Bytes = 128 * K1 * 2;
    static constexpr uint32_t kTmemCols = 512;
    static constexpr uint32_t kColD2 = 256, kColD3 = 448;
    static constexpr uint32_t kIdescHalf = instr_desc_bf16(128, 128), kIdescOut = instr_desc_bf16(128, NO);

    // tanh(D + bias) of the 128 TMEM columns [src, src+128) -> bf16 pairs in [dst, dst+64); bias points at the half's first column.
    // `tlane` = TMEM address of this warp's lane quarter at column 0 of the allocation.
    static __device__ __forceinline__ void half_epilogue(uint32_t tlane, uint32_t src, uint32_t dst, const float *bias)
    {
        uint32_t v[2][32];
        tmem_ld32(tlane + src, v[0]);
#pragma unroll
        for (int j = 0; j < 4; j++) {
            uint32_t o[16];
            tc_wait_ld();
            if (j + 1 < 4) tmem_ld32(tlane + src + 32 * (j + 1), v[(j + 1) & 1]);   // flies while chunk j is processed
#pragma unroll
            for (int i = 0; i < 16; i++) {
                const float2 b = *reinterpret_cast<const float2 *>(bias + 32 * j + 2 * i);
                const float2 y = fadd2(v[j & 1][2 * i], v[j & 1][2 * i + 1], b);
                o[i] = pack_bf16(tanh_approx(y.x), tanh_approx(y.y));
            }
            tmem_st16(tlane + dst + 16 * j, o);
        }
        tc_wait_st();
    }

    // ---- UMMA issue: called by ONE CONVERGED WARP, one elected lane issues.  Layer 1 (SS): A1 in shared memory (canonical [128][K1]) x W1 -> D1, two halves.
    // `narrow` (a net with 128 hidden units on this 256-wide kernel): the units are the first N-half of every layer and the
    // first half of the next layer's K, so only half a of layers 1 and 2 and 8 of the 16 K-steps of layers 2 and 3 are issued
    // (the other halves of the padded image are zeros and would add exactly nothing).
    static __device__ __forceinline__ void issue_l1(const uint8_t *image, const uint8_t *a1, uint32_t tmem_base, uint64_t *bar_a, uint64_t *bar_b, bool narrow)
    {
        tc_fence_after();
        const uint32_t sa = smem_u32(a1), sb = smem_u32(image + kW1);
        if (elect_one()) {
#pragma unroll
            for (int h = 0; h < 2; h++) {
                if (h == 1 && narrow) break;
#pragma unroll
                for (int k = 0; k < K1 / 16; k++)
                    umma_ss(tmem_base + 128 * h, smem_desc(sa + k * 2 * 128 * 16, 128 * 16, 128),
                            smem_desc(sb + k * 2 * H * 16 + h * 128 * 16, H * 16, 128), kIdescHalf, k > 0);
                umma_commit(h ? bar_b : bar_a);
            }
        }
        __syncwarp();
    }
    // Layer 2 (TS): A2 (TMEM cols [0,128), 8 columns per K-chunk) x W2 -> D2 = [256,512), two N-halves
    static __device__ __forceinline__ void issue_l2(const uint8_t *image, uint32_t tmem_base, uint64_t *bar_a, uint64_t *bar_b, bool narrow)
    {
        tc_fence_after();
        const uint32_t sb = smem_u32(image + kW2);
        if (elect_one()) {
#pragma unroll
            for (int h = 0; h < 2; h++) {
                if (h == 1 && narrow) break;
#pragma unroll
                for (int k = 0; k < H / 16; k++)
                    if (!(narrow && k >= H / 32)) umma_ts(tmem_base + kColD2 + 128 * h, tmem_base + 8 * k, smem_desc(sb + k * 2 * H * 16 + h * 128 * 16, H * 16, 128), kIdescHalf, k > 0);
                umma_commit(h ? bar_b : bar_a);
            }
        }
        __syncwarp();
    }
    // Layer 3 (TS): A3 (K-chunks 0-7 at [256,320), 8-15 at [384,448)) x W3 -> D3 = [448,448+NO)
    static __device__ __forceinline__ void issue_l3(const uint8_t *image, uint32_t tmem_base, uint64_t *bar, bool narrow)
    {
        tc_fence_after();
        const uint32_t sb = smem_u32(image + kW3);
        if (elect_one()) {
#pragma unroll
            for (int k = 0; k < H / 16; k++)
                if (!(narrow && k >= H / 32)) umma_ts(tmem_base + kColD3, tmem_base + kColD2 + (k < 8 ? 8 * k : 128 + 8 * (k - 8)), smem_desc(sb + k * 2 * NO * 16, NO * 16, 128), kIdescOut, k > 0);
            umma_commit(bar);
        }
        __syncwarp();
    }
    // one output of this thread's row, column `o` chosen at run time (the value head sits at 3N): D3[o] + b3[o]
    static __device__ __forceinline__ float load_output(const uint8_t *image, uint32_t tlane, uint32_t o)
    {
        const float *bias = reinterpret_cast<const float *>(image + kBias);
        const uint32_t v = tmem_ld1(tlane + kColD3 + o);
        tc_wait_ld();
        return __uint_as_float(v) + bias[2 * H + o];
    }
    // logits of this thread's row: D3 + b3
    static __device__ __forceinline__ void load_logits(const uint8_t *image, uint32_t tlane, float (&logit)[NO])
    {
        const float *bias = reinterpret_cast<const float *>(image + kBias);
#pragma unroll
        for (int j = 0; j < NO / 16; j++) {
            uint32_t v[16];
            tmem_ld16(tlane + kColD3 + 16 * j, v);
            tc_wait_ld();
#pragma unroll
            for (int i = 0; i < 16; i += 2) {
                const float2 y = fadd2(v[i], v[i + 1], *reinterpret_cast<const float2 *>(bias + 2 * H + 16 * j + i));
                logit[16 * j + i] = y.x; logit[16 * j + i + 1] = y.y;
            }
        }
    }
};

// named barrier over `n` threads (ids 1.. ; 0 is __syncthreads)
__device__ __forceinline__ void bar_sync(uint32_t id, uint32_t n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_arrive(uint32_t id, uint32_t n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

}  // namespace tc
}  // namespace im
