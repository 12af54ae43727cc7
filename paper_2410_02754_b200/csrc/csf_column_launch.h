// csf_column_launch.h — per-order launchers of the column kernel (defined in csf_column_p.cu, one object per order).
#pragma once
#include <cuda_runtime.h>
#include <cstddef>

namespace csf {

struct ColParams;
struct ColInfo { int lanes; size_t smem; };    // real lanes per CTA (4 per spinor vector), dynamic shared memory

#define CSF_DECL_COL(P) \
    cudaError_t launch_column_p##P(int ks, int mode, bool f32, const ColParams& cp, long long nblocks, cudaStream_t s); \
    ColInfo column_info_p##P();
CSF_DECL_COL(1) CSF_DECL_COL(2) CSF_DECL_COL(3) CSF_DECL_COL(4) CSF_DECL_COL(5) CSF_DECL_COL(6) CSF_DECL_COL(7)
#undef CSF_DECL_COL
// wide variant of the cell-per-iteration kernel (8 vectors per CTA), orders 4 and 5
#define CSF_DECL_COLWIDE(P) \
    cudaError_t launch_column_wide_p##P(int ks, int mode, bool f32, const ColParams& cp, long long nblocks, cudaStream_t s); \
    ColInfo column_info_wide_p##P();
CSF_DECL_COLWIDE(4) CSF_DECL_COLWIDE(5)
#undef CSF_DECL_COLWIDE
// wide kernel of order 5 with two gather warps (fused projector gather of another block, ColParams::g; FP64, KS = 5)
cudaError_t launch_column_wide_p5_g(int ks, int mode, bool f32, const ColParams& cp, long long nblocks, cudaStream_t s);
ColInfo column_info_wide_p5_g();
// warp-specialised kernel (csf_colws.cuh: 8 vectors per CTA, persistent CTAs), orders 4 and 5
#define CSF_DECL_COLW(P) \
    cudaError_t launch_column_ws_p##P(int ks, int mode, bool f32, const ColParams& cp, int nctas, cudaStream_t s); \
    ColInfo column_info_ws_p##P();
CSF_DECL_COLW(4) CSF_DECL_COLW(5)
#undef CSF_DECL_COLW

}  // namespace csf
