// csf_colws_p.cu — instantiates the warp-specialised column kernel (csf_colws.cuh) for one FE order
// (compile with -DCSF_P=4 or 5); one translation unit per order so that the orders build in parallel.
#include "csf_colws.cuh"
#include "csf_column_launch.h"

#ifndef CSF_P
#error "compile with -DCSF_P=<order>"
#endif

#define CSF_CAT2(a, b) a##b
#define CSF_CAT(a, b) CSF_CAT2(a, b)
#define CSF_FN(name) CSF_CAT(CSF_CAT(name, _ws_p), CSF_P)

namespace csf {

namespace {

template <typename T, int KS, int MODE>
cudaError_t launch_t(const ColParams& cp, int nctas, cudaStream_t s) {
    // the opt-in to > 48 KB of dynamic shared memory belongs to the device's context: remember it per device
    static bool configured[64] = {};
    auto kern = colws_kernel<T, CSF_P, KS, MODE>;
    using Cfg = WsCfg<T, CSF_P>;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    kern<<<(unsigned)nctas, Cfg::NT, Cfg::SMEM, s>>>(cp);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_real(int ks, int mode, const ColParams& cp, int nctas, cudaStream_t s) {
    if (ks <= 5) return mode == 2 ? launch_t<T, 5, 2>(cp, nctas, s) : mode == 1 ? launch_t<T, 5, 1>(cp, nctas, s) : launch_t<T, 5, 0>(cp, nctas, s);
    return mode == 2 ? launch_t<T, 8, 2>(cp, nctas, s) : mode == 1 ? launch_t<T, 8, 1>(cp, nctas, s) : launch_t<T, 8, 0>(cp, nctas, s);
}
}  // namespace

cudaError_t CSF_FN(launch_column)(int ks, int mode, bool f32, const ColParams& cp, int nctas, cudaStream_t s) {
    return f32 ? launch_real<float>(ks, mode, cp, nctas, s) : launch_real<double>(ks, mode, cp, nctas, s);
}

ColInfo CSF_FN(column_info)() { return ColInfo{kWsLanes, WsCfg<double, CSF_P>::SMEM}; }

}  // namespace csf
