// pipe_ptx.cuh -- PTX wrappers shared by the pipelined slice-step kernels (mbarrier, TMA bulk copy, cp.async).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace prism {

// ---- PTX helpers ------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count)
{ asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory"); }
__device__ __forceinline__ void mbar_fence_init()
{ asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes)
{ asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory"); }
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity)
{
    const unsigned addr = smem_u32(bar);
    unsigned done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(addr), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gmem_src, unsigned bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src)
{ asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(gmem_src) : "memory"); }
__device__ __forceinline__ void cp_async_arrive(uint64_t* bar)
{ asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory"); }
__device__ __forceinline__ void named_barrier(int id, int nthreads)
{ asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }

// ---- programmatic dependent launch (PDL) ------------------------------------------------------------------
// The slice loop is a chain of kernels in one stream, each consuming what the previous one wrote.  Launched with
// the programmatic-stream-serialization attribute, the next kernel's launch is prepared while the current one
// runs and its CTAs start as soon as the last CTA of the current one has exited; griddep_wait() then blocks until
// the previous grid has completed and its writes are visible.  Every kernel of the chain calls griddep_wait()
// before touching global data, so "the previous kernel has completed" still implies all earlier ones have.
// No kernel triggers its dependents early (griddepcontrol.launch_dependents): measured on the B200, an early
// trigger keeps the launch-bound gain (MS2 32.0 k -> 36.2 k probes/s either way) but makes the HBM-bound passes
// slower -- 2048^2 x 1201 beams x 24 slices: 845 ms with the trigger at the top of every kernel, 745 ms without
// (and 746 ms with plain stream order); P8 165.9 -> 164.7 ms per step.
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <class... KArgs, class... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t stream,
                              Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

constexpr int PIPE_SMEM_MAX = 227 * 1024;
constexpr int PIPE_HEADER = 1024;                     // mbarriers
__host__ __device__ constexpr int round_up_c(int a, int b) { return (a + b - 1) / b * b; }
// band of a grid with square pixels: |k| <= floor(N / 3), rounded up to 32 columns
template <int N> struct DefaultBand { static constexpr int XB = (N / 3 + 1 + 31) / 32 * 32; };

int num_sms();

}  // namespace prism
