// generals_variant.cu -- one kernel instantiation per translation unit: compile with -DGEN_VARIANT_ID=n
// (n indexes GEN_VARIANTS of generals_variants.h).
#include "generals_variants.h"

#ifndef GEN_VARIANT_ID
#error "compile with -DGEN_VARIANT_ID=<n>"
#endif

namespace gen {

template <int ID> struct Sel;
#define GEN_DEFINE(id, np, h, w, ff)                                    \
    template <> struct Sel<id> {                                        \
        static constexpr int NP = np, H = h, W = w;                     \
        static constexpr uint32_t FF = ff;                              \
    };
GEN_VARIANTS(GEN_DEFINE)
#undef GEN_DEFINE

#define GEN_CAT_(a, b) a##b
#define GEN_CAT(a, b) GEN_CAT_(a, b)

cudaError_t GEN_CAT(launch_variant_, GEN_VARIANT_ID)(const KParams &kp, int grid, int block, size_t smem,
                                                     cudaStream_t stream) {
    using S = Sel<GEN_VARIANT_ID>;
    auto kernel = k_generals<S::NP, S::H, S::W, S::FF>;
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    kernel<<<grid, block, smem, stream>>>(kp);
    return cudaGetLastError();
}

}  // namespace gen
