// csf_column_p.cu — instantiates the column kernel for one FE order (compile with -DCSF_P=<1..7>); one translation
// unit per order so that the orders build in parallel.
#include "csf_column.cuh"
#include "csf_column_launch.h"

#ifndef CSF_P
#error "compile with -DCSF_P=<order>"
#endif

#define CSF_CAT2(a, b) a##b
#define CSF_CAT(a, b) CSF_CAT2(a, b)

namespace csf {

namespace {
#ifdef CSF_WIDE
// wide variant (its own translation unit, orders 4 and 5): 8 vectors per CTA, 128-byte row pieces, a main warp = one plane
constexpr int kLanes = 32;
#define CSF_FN(name) CSF_CAT(CSF_CAT(name, _wide_p), CSF_P)
#else
constexpr int kLanes = CSF_P <= 6 ? 16 : 8;      // order 7 does not fit shared memory with 4 vectors per CTA
#define CSF_FN(name) CSF_CAT(CSF_CAT(name, _p), CSF_P)
#endif

#ifdef CSF_GATHERW
constexpr int kGatherWarps = CSF_GATHERW;        // translation unit of the kernels with gather warps (FP64, KS = 5 only)
#else
constexpr int kGatherWarps = 0;
#endif

template <typename T, int KS, int MODE>
cudaError_t launch_t(const ColParams& cp, long long nblocks, cudaStream_t s) {
    // the opt-in to > 48 KB of dynamic shared memory belongs to the device's context: remember it per device
    static bool configured[64] = {};
    auto kern = column_kernel<T, CSF_P, KS, MODE, kLanes, col_aux_warps(CSF_P, sizeof(T) == 4, MODE, kLanes), kGatherWarps>;
    using Cfg = ColCfg<T, CSF_P, kLanes, col_aux_warps(CSF_P, sizeof(T) == 4, MODE, kLanes), kGatherWarps>;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    kern<<<(unsigned)nblocks, Cfg::NT, Cfg::SMEM, s>>>(cp);
    return cudaGetLastError();
}

// (inside the unnamed namespace: every order's translation unit instantiates launch_real<T>, and with external linkage
// the linker would keep one of them for all orders)
template <typename T>
cudaError_t launch_real(int ks, int mode, const ColParams& cp, long long nblocks, cudaStream_t s) {
    if (ks <= 5) return mode == 2 ? launch_t<T, 5, 2>(cp, nblocks, s) : mode == 1 ? launch_t<T, 5, 1>(cp, nblocks, s) : launch_t<T, 5, 0>(cp, nblocks, s);
    return mode == 2 ? launch_t<T, 8, 2>(cp, nblocks, s) : mode == 1 ? launch_t<T, 8, 1>(cp, nblocks, s) : launch_t<T, 8, 0>(cp, nblocks, s);
}
}  // namespace

#ifdef CSF_GATHERW
// column step + fused projector gather of another block (ColParams::g): complex128 blocks, 18 projectors per atom (KS = 5)
cudaError_t CSF_CAT(CSF_FN(launch_column), _g)(int ks, int mode, bool f32, const ColParams& cp, long long nblocks, cudaStream_t s) {
    if (f32 || ks != 5) return cudaErrorInvalidValue;
    return mode == 2 ? launch_t<double, 5, 2>(cp, nblocks, s) : mode == 1 ? launch_t<double, 5, 1>(cp, nblocks, s) : launch_t<double, 5, 0>(cp, nblocks, s);
}

ColInfo CSF_CAT(CSF_FN(column_info), _g)() { return ColInfo{kLanes, ColCfg<double, CSF_P, kLanes, col_aux_warps(CSF_P, false, 2, kLanes), kGatherWarps>::SMEM}; }
#else
cudaError_t CSF_FN(launch_column)(int ks, int mode, bool f32, const ColParams& cp, long long nblocks, cudaStream_t s) {
    return f32 ? launch_real<float>(ks, mode, cp, nblocks, s) : launch_real<double>(ks, mode, cp, nblocks, s);
}

ColInfo CSF_FN(column_info)() { return ColInfo{kLanes, ColCfg<double, CSF_P, kLanes>::SMEM}; }
#endif

}  // namespace csf
