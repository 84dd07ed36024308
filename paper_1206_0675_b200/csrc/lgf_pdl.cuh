// lgf_pdl.cuh -- programmatic dependent launch (sm_90+) for the kernels of one iteration: they are launched
// with the programmatic-stream-serialization attribute, and every kernel begins with pdl_enter(), which waits
// until the preceding kernel in the stream has completed and its writes are visible (griddepcontrol.wait) --
// nothing a kernel reads may be touched before it, not even the stop flag.  The next kernel is released as this
// one's blocks exit (the implicit trigger), so its launch latency and block scheduling overlap this kernel's
// tail instead of following its completion.  One iteration has five kernel boundaries; measured on B200 (whole
// iteration, off -> on): 8^4 0.0260 -> 0.0173 ms, 16^4 0.0450 -> 0.0340, 32^4 fp32/18 0.2185 -> 0.2071, 32^4
// fp64/18 0.378 -> 0.369, 64^4 6.71 -> 6.66 -- it does for the launch-bound small lattices what capturing the
// iteration in a CUDA graph was meant to do, and works on every stream, the legacy default stream included
// (where stream capture is not allowed).
// NOT used: an explicit early trigger (griddepcontrol.launch_dependents at the top of every block).  It lets
// the dependent grid's blocks become resident, spinning at their wait with their registers and shared memory
// allocated, while the primary grid still has waves to run: 32^4 fp64 0.377 -> 0.400 ms, 64^4 6.65 -> 8.35 ms.
// A kernel launched the ordinary way sees the wait as a no-op.  Part of liblgf (CUDA path).
#pragma once
#include <cuda_runtime.h>

#include <mutex>
#include <tuple>
#include <vector>

namespace lgf {

__device__ __forceinline__ void pdl_enter() {
#if defined(__CUDA_ARCH__) && __CUDA_ARCH__ >= 900
    cudaGridDependencySynchronize();
#endif
}

// Opt a kernel in to more than 48 KB of dynamic shared memory ONCE per (kernel, device), not on every launch: the
// attribute call is a runtime round trip, and the small lattices are launch-bound.
template <class K>
cudaError_t ensure_dynamic_smem(K kern, size_t bytes) {
    if (bytes <= 48 * 1024) return cudaSuccess;
    static std::mutex mu;
    static std::vector<std::tuple<const void *, int, size_t>> seen;
    int dev = 0;
    cudaGetDevice(&dev);
    const void *key = reinterpret_cast<const void *>(kern);
    std::lock_guard<std::mutex> lock(mu);
    for (auto &e : seen)
        if (std::get<0>(e) == key && std::get<1>(e) == dev) {
            if (std::get<2>(e) >= bytes) return cudaSuccess;
            const cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
            if (err == cudaSuccess) std::get<2>(e) = bytes;
            return err;
        }
    const cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (err == cudaSuccess) seen.emplace_back(key, dev, bytes);
    return err;
}

// A stream plus the context's programmatic-dependent-launch setting (lgf_tune "pdl", per context).  Converts from
// and to cudaStream_t, so launchers that do not care keep passing a plain stream (dependent launch allowed).
struct LaunchStream {
    cudaStream_t s;
    bool pdl;
    LaunchStream(cudaStream_t stream = nullptr, bool allow = true) : s(stream), pdl(allow) {}
    operator cudaStream_t() const { return s; }
};

// kernel<<<grid, block, smem, stream>>>(args...) with the attribute that lets it start while its predecessor drains
template <class... KArgs, class... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, LaunchStream stream, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream.s;
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr.val.programmaticStreamSerializationAllowed = stream.pdl ? 1 : 0;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

}  // namespace lgf
