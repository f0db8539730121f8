// generals_variant.cu -- one kernel instantiation per translation unit: compile with -DGEN_VARIANT_ID=n
// (n indexes GEN_VARIANTS of generals_variants.h).
#include <atomic>

#include "generals_variants.h"

#ifndef GEN_VARIANT_ID
#error "compile with -DGEN_VARIANT_ID=<n>"
#endif

namespace gen {

template <int ID> struct Sel;
#define GEN_DEFINE(id, kind, np, h, w, ff, maxt, minb)                  \
    template <> struct Sel<id> {                                        \
        static constexpr int KIND = kind, NP = np, H = h, W = w;        \
        static constexpr uint32_t FF = ff;                              \
        static constexpr int MAXT = maxt, MINB = minb;                  \
    };
GEN_VARIANTS(GEN_DEFINE)
#undef GEN_DEFINE

template <typename S, int KIND> struct KernelOf;
template <typename S> struct KernelOf<S, 0> {
    static constexpr auto fn = k_generals<S::NP, S::H, S::W, S::FF, false>;
};
template <typename S> struct KernelOf<S, 1> {
    static constexpr auto fn = k_step<S::NP, S::H, S::W, S::MAXT, S::MINB, false, (S::FF != 0)>;
};
template <typename S> struct KernelOf<S, 2> {   // kinds 2 / 3: the same kernels with the official generator (R36)
    static constexpr auto fn = k_generals<S::NP, S::H, S::W, S::FF, true>;
};
template <typename S> struct KernelOf<S, 3> {
    static constexpr auto fn = k_step<S::NP, S::H, S::W, S::MAXT, S::MINB, true, false>;
};

#define GEN_CAT_(a, b) a##b
#define GEN_CAT(a, b) GEN_CAT_(a, b)

cudaError_t GEN_CAT(launch_variant_, GEN_VARIANT_ID)(const KParams &kp, int grid, int block, size_t smem,
                                                     cudaStream_t stream) {
    using S = Sel<GEN_VARIANT_ID>;
    auto kernel = KernelOf<S, S::KIND>::fn;
    // the opt-in for more than 48 KB of dynamic shared memory is per device: one flag per device ordinal
    static std::atomic<unsigned long long> attr_set{0};
    int dev = 0;
    if (cudaError_t e = cudaGetDevice(&dev); e != cudaSuccess) return e;
    const unsigned long long bit = 1ull << (dev & 63);
    if (dev >= 64 || !(attr_set.load(std::memory_order_acquire) & bit)) {
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem);
        if (e != cudaSuccess) return e;
        attr_set.fetch_or(bit, std::memory_order_release);
    }
    // Programmatic dependent launch: the CTAs of this grid may be placed while the previous grid in the stream
    // drains; both kernels execute griddepcontrol.wait before their first global access, so the overlap is
    // launch latency and prologue only.
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, kp);
}

}  // namespace gen

#ifdef GEN_TRACE  // development only
extern "C" int GEN_CAT(gen_debug_trace_, GEN_VARIANT_ID)(unsigned long long *out, int n) {
    cudaMemcpyFromSymbol(out, gen::g_trace, sizeof(unsigned long long) * (size_t)n);
    void *p = nullptr;
    cudaGetSymbolAddress(&p, gen::g_trace);
    cudaMemset(p, 0, sizeof(gen::g_trace));
    return 0;
}
#endif
