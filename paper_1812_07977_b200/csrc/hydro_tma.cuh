// hydro_tma.cuh -- TMA (cp.async.bulk.tensor) + mbarrier plumbing for the fused stage kernel.
//
// The padded SoA state U[v][K][J][I] is described to the TMA unit as a rank-4
// tensor (I, J, K, v); one instruction brings the (tile + 2-cell halo) box of one z-plane for all
// five conserved variables into shared memory and signals an mbarrier.  Ghost layers exist
// physically (TMA cannot mirror or wrap); boxes that run past the padded extents are zero-filled
// by the hardware and feed only threads that never store.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>

namespace hyd {
namespace tma {

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}

__device__ __forceinline__ void fence_barrier_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

// L2 prefetch of the 128-byte line that holds `p`: one instruction for the lanes that call it, no destination,
// nothing to wait for (stage 2 warms the lines its plain U0 loads will read a plane later).  The bulk form
// (cp.async.bulk.prefetch.L2 = UBLKPF.L2) takes uniform-register operands: the compiler wraps it in a loop
// over the active lanes, seven instructions per lane -- measured slower than this per-lane form.
__device__ __forceinline__ void prefetch_l2_line(const void *p)
{
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p) : "memory");
}

// generic-proxy accesses before, async-proxy (TMA) accesses after
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}

__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}

// Wait on a block-wide hand-off barrier: try_wait with a suspend-time hint, so that a warp that finds the
// phase incomplete is parked by the hardware for up to ~200 ns instead of re-polling at once (measured:
// the flux barrier is polled 29 times per warp and plane without the hint; with it 256^3 runs 1.5 % and
// 128^3 2 % faster).  The TMA waits keep the plain form: the data has almost always landed.
#ifndef HYD_WAIT_HINT
#define HYD_WAIT_HINT 200
#endif
__device__ __forceinline__ void mbar_wait_sync(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1, %2;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(smem_u32(bar)), "r"(parity), "r"((uint32_t)HYD_WAIT_HINT)
        : "memory");
}

// one rank-4 box: coordinates (c0 fastest) -> shared memory at dst, completion on bar
__device__ __forceinline__ void load_4d(void *dst, const CUtensorMap *map, int c0, int c1, int c2, int c3,
                                        uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(smem_u32(dst)), "l"((unsigned long long)map), "r"(c0), "r"(c1), "r"(c2), "r"(c3),
        "r"(smem_u32(bar))
        : "memory");
}

// ---- host side ---------------------------------------------------------------------------

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

// cuTensorMapEncodeTiled through the runtime's driver entry point (no -lcuda)
inline EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

// Tensor map of one padded 5-variable fp64 state: dims (px, Ny, Nz, 5), strides in doubles
// (px, sy, sv); box (bx, by, 1, 5).
inline bool make_state_map(CUtensorMap *map, const double *base, int px, int Ny, int Nz, long long sy,
                           long long sv, int bx, int by)
{
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return false;
    const cuuint64_t dims[4] = { (cuuint64_t)px, (cuuint64_t)Ny, (cuuint64_t)Nz, 5 };
    const cuuint64_t strides[3] = { (cuuint64_t)px * 8, (cuuint64_t)sy * 8, (cuuint64_t)sv * 8 };
    const cuuint32_t box[4] = { (cuuint32_t)bx, (cuuint32_t)by, 1, 5 };
    const cuuint32_t estr[4] = { 1, 1, 1, 1 };
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void *)base, dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace tma
}  // namespace hyd
