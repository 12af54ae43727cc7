// csf_api.cu — C ABI of libcsf (see include/csf.h): context, host-side preprocessing, launch sequencing.
#include "../../include/csf.h"
#include "csf_kernels.cuh"
#include "csf_column.cuh"
#include "csf_colws.cuh"
#include "csf_subspace.cuh"
#include "csf_dense.cuh"
#include "csf_column_launch.h"
#include "csf_tables.h"

#include <cuda.h>
#include <cusolverDn.h>
#include <dlfcn.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <numeric>
#include <string>
#include <vector>

using namespace csf;

namespace {

thread_local std::string g_create_error;

struct DevBuf {
    void* p = nullptr; size_t bytes = 0;
    ~DevBuf() { release(); }
    void release() { if (p) cudaFree(p); p = nullptr; bytes = 0; }
    cudaError_t alloc(size_t n) { release(); if (n == 0) return cudaSuccess; cudaError_t e = cudaMalloc(&p, n); if (e == cudaSuccess) bytes = n; return e; }
    template <class T> cudaError_t upload(const std::vector<T>& v) {
        cudaError_t e = alloc(std::max<size_t>(v.size(), 1) * sizeof(T)); if (e != cudaSuccess) return e;
        return v.empty() ? cudaSuccess : cudaMemcpy(p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice);
    }
    template <class T> T* as() const { return static_cast<T*>(p); }
};

}  // namespace

struct csf_ctx {
    int device = 0; cudaStream_t stream = nullptr;
    int ncell[3], bc[3], p = 0, n = 0;
    double box[3], h[3];
    int nfree[3]; long long M = 0; int E = 0;
    Gll1D gll; Dir1D dir[3];
    bool have_pot = false;
    DevBuf d_col_order, d_vb;
    double kpt[3] = {0.0, 0.0, 0.0}; bool kpt_on = false;      // Bloch vector of csf_set_kpoint (dense path only)
    bool proj_complex = false; DevBuf d_g_pack_im, d_gk;         // Im P~ (csf_set_projectors_complex); S sum_d k_d G_d^(e) S in fragment order
    DevBuf d_cellmat; int dense_nq = 0, dense_n3p = 0;      // cell matrices of csf_set_potential_quadrature (fragment order, csf_dense.cuh)
    DevBuf d_inv_mass, d_occ;               // 1 / m_I (csf_density), occupation numbers of the last csf_density call
    DevBuf d_sub_ptr[kColMaxAuxWarps - 1], d_sub_desc[kColMaxAuxWarps - 1], d_a_pack[kColMaxAuxWarps - 1], d_ent_locf;     // [nq - 2]: nq expansion warps per CTA
    int seg_len = 0, chunk_group = 16;      // cells per z-segment (0 = the kernel's default), vector chunks scheduled back to back (csf_set_tuning)
    int lanes_force = 0;                    // CSF_LANES=16|32 pins the column kernel variant (tests, sweeps); 0 = measured policy
    int kernel_force = 0;                   // CSF_KERNEL=wide|ws pins the 8-vector kernel of orders 4 and 5 (1 | 2)
    bool bulk_gather = true;                // CSF_GATHER=reg pins the register-load projector gather (tests run both)
    int fused_gather = -1;                  // CSF_FUSED_GATHER=0|1: csf_filter's fused half-block path off | on for every block size; -1 = policy
    // projectors
    int natoms = 0, npj_uniform = 0, npjp = 0; long long crows = 0;
    DevBuf d_ent_node, d_atom_coff, d_atom_npj, d_atom_type, d_delta, d_delta_ptr, d_gb_atom, d_gb_beg, d_gb_end, d_gb_k0, d_g_pack;
    int n_gather_blocks = 0;
    int variant = 0;
    long long launches = 0;
    int sm_count = 148; size_t smem_optin = 0;
    std::string err;
    // csf_filter_host: two (x, y) column-chunk slots + one workspace, copy streams and events
    DevBuf h_x[2], h_y[2], h_w;
    cudaStream_t hs_in = nullptr, hs_out = nullptr;
    cudaEvent_t ev_in[2] = {nullptr, nullptr}, ev_cmp[2] = {nullptr, nullptr}, ev_out[2] = {nullptr, nullptr};
    int host_chunk = 64;
    // per-kernel-kind CUDA-event timing (csf_profile_*)
    bool prof = false;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof_ev[CSF_NKINDS];
    ~csf_ctx() {
        for (auto& v : prof_ev) for (auto& pr : v) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
        for (int s = 0; s < 2; ++s) { if (ev_in[s]) cudaEventDestroy(ev_in[s]); if (ev_cmp[s]) cudaEventDestroy(ev_cmp[s]); if (ev_out[s]) cudaEventDestroy(ev_out[s]); }
        if (hs_in) cudaStreamDestroy(hs_in);
        if (hs_out) cudaStreamDestroy(hs_out);
    }
};

namespace {

int fail(csf_ctx* c, int code, const std::string& msg) { if (c) c->err = msg; else g_create_error = msg; return code; }
int cuda_fail(csf_ctx* c, cudaError_t e, const char* what) { return fail(c, CSF_ECUDA, std::string(what) + ": " + cudaGetErrorString(e)); }
#define CSF_CUDA(ctx, call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return cuda_fail(ctx, e__, #call); } while (0)
// nothing may throw across the C ABI (csf.h): every entry point that allocates host memory runs inside this guard
#define CSF_GUARD_BEGIN try {
#define CSF_GUARD_END(ctx) } catch (const std::bad_alloc&) { return fail(const_cast<csf_ctx*>(ctx), CSF_ENOMEM, "out of host memory"); } \
                           catch (...) { return fail(const_cast<csf_ctx*>(ctx), CSF_ECUDA, "unexpected C++ exception"); }

// brackets one kernel launch with two events when profiling is on
struct ProfScope {
    csf_ctx* c; int kind; cudaEvent_t e0 = nullptr, e1 = nullptr;
    ProfScope(csf_ctx* c_, int kind_) : c(c_), kind(kind_) {
        if (!c->prof) return;
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) { e0 = e1 = nullptr; return; }
        cudaEventRecord(e0, c->stream);
    }
    ~ProfScope() { if (e1) { cudaEventRecord(e1, c->stream); c->prof_ev[kind].push_back({e0, e1}); } }
};

bool have_wide(int p) { return p == 4 || p == 5; }

// kind: 0 = 4 vectors per CTA, 1 = 8 vectors per CTA (orders 4, 5), 2 = warp-specialised streaming kernel (orders 4, 5)
cudaError_t launch_column(int p, int ks, int mode, bool f32, int kind, const ColParams& cp, long long nblocks, cudaStream_t s) {
    if (kind == 2 && p == 4) return launch_column_ws_p4(ks, mode, f32, cp, (int)nblocks, s);
    if (kind == 2 && p == 5) return launch_column_ws_p5(ks, mode, f32, cp, (int)nblocks, s);
    if (kind == 1 && p == 4) return launch_column_wide_p4(ks, mode, f32, cp, nblocks, s);
    if (kind == 1 && p == 5) return launch_column_wide_p5(ks, mode, f32, cp, nblocks, s);
    switch (p) {
        case 1: return launch_column_p1(ks, mode, f32, cp, nblocks, s);
        case 2: return launch_column_p2(ks, mode, f32, cp, nblocks, s);
        case 3: return launch_column_p3(ks, mode, f32, cp, nblocks, s);
        case 4: return launch_column_p4(ks, mode, f32, cp, nblocks, s);
        case 5: return launch_column_p5(ks, mode, f32, cp, nblocks, s);
        case 6: return launch_column_p6(ks, mode, f32, cp, nblocks, s);
        case 7: return launch_column_p7(ks, mode, f32, cp, nblocks, s);
    }
    return cudaErrorInvalidValue;
}

ColInfo column_info(int p, int kind) {
    if (kind == 2 && p == 4) return column_info_ws_p4();
    if (kind == 2 && p == 5) return column_info_ws_p5();
    if (kind == 1 && p == 4) return column_info_wide_p4();
    if (kind == 1 && p == 5) return column_info_wide_p5();
    switch (p) {
        case 1: return column_info_p1(); case 2: return column_info_p2(); case 3: return column_info_p3(); case 4: return column_info_p4();
        case 5: return column_info_p5(); case 6: return column_info_p6(); default: return column_info_p7();
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link-time dependency on libcuda)
EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr; cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// FP64 tensor map of rank `rank`: dims / box in elements (innermost first), strides in bytes for dims 1..rank-1
bool encode_map(CUtensorMap* tm, const void* base, int rank, const cuuint64_t* dims, const cuuint64_t* strides, const cuuint32_t* box, bool f32 = false) {
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    cuuint32_t es[5] = {1, 1, 1, 1, 1};
    return fn(tm, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, (cuuint32_t)rank, const_cast<void*>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

size_t ctp_bytes(const csf_ctx* c, int nvec);
size_t f32_block_bytes(const csf_ctx* c, int nvec);

// kernel mode for a block of nvec vectors with vpc vectors per CTA. 2: periodic cubic-cell mesh, full vector chunks;
// 1: x, y periodic, full chunks (z and the cell shape general); 0: general
int column_mode(const csf_ctx* c, int nvec, int vpc, bool f32) {
    if (!(c->bc[0] == CSF_BC_PERIODIC && c->bc[1] == CSF_BC_PERIODIC && nvec % vpc == 0 && c->variant != 1)) return 0;
    const bool cubic = c->h[0] * c->h[0] / (c->h[1] * c->h[1]) == 1.0 && c->h[0] * c->h[0] / (c->h[2] * c->h[2]) == 1.0;
    // mode 1 measured slower than 0 for the narrow FP64 kernel
    return (c->bc[2] == CSF_BC_PERIODIC && cubic) ? 2 : ((f32 || vpc == 8) ? 1 : 0);
}

// Which column kernel runs (kind): orders 4 and 5 take a kernel with 8 vectors per CTA — the cell-per-iteration kernel
// (kind 1, csf_column.cuh) or the warp-specialised streaming kernel (kind 2, csf_colws.cuh) —, the other orders the
// cell-per-iteration kernel with 4 vectors per CTA (kind 0). CSF_LANES=16 pins kind 0, CSF_KERNEL=ws|wide pins 2 | 1 (tests, sweeps).
int column_kind(const csf_ctx* c) {
    if (!have_wide(c->p) || c->lanes_force == 16) return 0;
    const bool ws_ok = c->ncell[0] < 32768 && c->ncell[1] < 32768;       // (the kernel packs cx, cy into 16 bits each)
    if (c->kernel_force == 2 && ws_ok) return 2;
    if (c->kernel_force == 1) return 1;
    return 1;
}
int aux_warps(const csf_ctx* c, bool f32, int mode, int kind) { return kind == 2 ? kWsRoleWarps : col_aux_warps(c->p, f32, mode, kind == 1 ? 32 : 16); }

// What a column launch of the fused path carries for its gather warps: the block whose coefficients C = P~^T src they compute
struct FusedGather { const void* src; long long ld; int nvec; double* dC; };

// a5: C = P~^T src (cleared first) as a kernel of its own
int enqueue_gather(csf_ctx* c, const void* src, long long ld, int nvec, double* dC, bool f32) {
    const long long ldc = nvec;
    {
        CSF_CUDA(c, cudaMemsetAsync(dC, 0, (size_t)c->crows * ldc * sizeof(double2), c->stream));
        GatherParams gp{};
        gp.src = src; gp.ld = ld; gp.nvec = nvec;
        gp.gb_atom = c->d_gb_atom.as<int>(); gp.gb_beg = c->d_gb_beg.as<int>(); gp.gb_end = c->d_gb_end.as<int>();
        gp.ent_node = c->d_ent_node.as<int>(); gp.g_pack = c->d_g_pack.as<double>(); gp.gb_k0 = c->d_gb_k0.as<int>();
        gp.atom_coff = c->d_atom_coff.as<long long>(); gp.atom_npj = c->d_atom_npj.as<int>();
        gp.C = dC; gp.ldc = ldc;
        dim3 gg(c->n_gather_blocks, (nvec + 16 * kGatherNT - 1) / (16 * kGatherNT));
        {
            ProfScope ps(c, CSF_KIND_PGATHER);
            // blocks with 16-byte aligned rows: the bulk-copy kernel (src staged in shared memory by cp.async.bulk); complex64
            // blocks have an even leading dimension (f32_block_bytes), so their rows qualify too
            const bool bulk = c->bulk_gather && ((uintptr_t)src & 15) == 0 && (!f32 || ld % 2 == 0);
            if (bulk) {
                static bool configured[64] = {};
                int dev = 0; CSF_CUDA(c, cudaGetDevice(&dev));
                if (dev < 0 || dev >= 64 || !configured[dev]) {
                    CSF_CUDA(c, cudaFuncSetAttribute(proj_gather_bulk_kernel<3, 2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kGbSmem));
                    CSF_CUDA(c, cudaFuncSetAttribute(proj_gather_bulk_kernel<3, 3, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kGbSmem));
                    CSF_CUDA(c, cudaFuncSetAttribute(proj_gather_bulk_kernel<4, 4, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kGbSmem));
                    CSF_CUDA(c, cudaFuncSetAttribute(proj_gather_bulk_kernel<3, 2, 2, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gb_smem<float>()));
                    CSF_CUDA(c, cudaFuncSetAttribute(proj_gather_bulk_kernel<3, 3, 0, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gb_smem<float>()));
                    CSF_CUDA(c, cudaFuncSetAttribute(proj_gather_bulk_kernel<4, 4, 0, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gb_smem<float>()));
                    if (dev >= 0 && dev < 64) configured[dev] = true;
                }
                if (f32) {
                    if (c->npj_uniform == 18) proj_gather_bulk_kernel<3, 2, 2, float><<<gg, 256, gb_smem<float>(), c->stream>>>(gp);
                    else if (c->npjp <= 24) proj_gather_bulk_kernel<3, 3, 0, float><<<gg, 256, gb_smem<float>(), c->stream>>>(gp);
                    else proj_gather_bulk_kernel<4, 4, 0, float><<<gg, 256, gb_smem<float>(), c->stream>>>(gp);
                }
                else if (c->npj_uniform == 18) proj_gather_bulk_kernel<3, 2, 2><<<gg, 256, kGbSmem, c->stream>>>(gp);
                else if (c->npjp <= 24) proj_gather_bulk_kernel<3, 3, 0><<<gg, 256, kGbSmem, c->stream>>>(gp);
                else proj_gather_bulk_kernel<4, 4, 0><<<gg, 256, kGbSmem, c->stream>>>(gp);
            }
            else if (c->npj_uniform == 18 && !f32) proj_gather_kernel<3, double, 2, 2><<<gg, 256, 0, c->stream>>>(gp);     // (slower than the full-DMMA form with float loads)
            else if (c->npjp <= 24) { if (f32) proj_gather_kernel<3, float><<<gg, 256, 0, c->stream>>>(gp); else proj_gather_kernel<3, double><<<gg, 256, 0, c->stream>>>(gp); }
            else { if (f32) proj_gather_kernel<4, float><<<gg, 256, 0, c->stream>>>(gp); else proj_gather_kernel<4, double><<<gg, 256, 0, c->stream>>>(gp); }
        }
        CSF_CUDA(c, cudaGetLastError());
        c->launches += 1;
    }
    return CSF_OK;
}

// a6: C~ = Delta C, written in the fragment order of the column kernel's DMMA B operand; clear_ct: the padding rows of C~
// must be zero (once per buffer and layout is enough)
int enqueue_delta(csf_ctx* c, const double* dC, double* dCt, int nvec, double sc, bool clear_ct = true) {
    const long long ldc = nvec;
    const int kind = column_kind(c); const bool ws = kind == 2;
    {
        DeltaParams dp{};
        const int lanes = column_info(c->p, kind).lanes, nchunks = (nvec + lanes / 4 - 1) / (lanes / 4);
        if (clear_ct) CSF_CUDA(c, cudaMemsetAsync(dCt, 0, ctp_bytes(c, nvec), c->stream));
        dp.C = reinterpret_cast<const double2*>(dC); dp.Ct = dCt; dp.ldc = ldc; dp.nvec = nvec;
        dp.lanes = lanes; dp.ks = c->npjp / 4; dp.nchunks = nchunks;
        dp.scale = ws ? sc : 1.0;          // the streaming kernel accumulates sc * (P~ C~) straight into its X tile
        dp.atom_coff = c->d_atom_coff.as<long long>(); dp.atom_npj = c->d_atom_npj.as<int>(); dp.atom_type = c->d_atom_type.as<int>();
        dp.delta = c->d_delta.as<double2>(); dp.delta_ptr = c->d_delta_ptr.as<long long>();
        dim3 dg(c->natoms, (nvec + 31) / 32);
        { ProfScope ps(c, CSF_KIND_DELTA); delta_apply_kernel<<<dg, 256, 0, c->stream>>>(dp); }
        CSF_CUDA(c, cudaGetLastError());
        c->launches += 1;
    }
    return CSF_OK;
}

// a1-a4, a7, a8: dst += sc * i^rot * (H_loc - shift + P~ C~) src; fg != nullptr: the launch also carries the projector
// gather of another block (wide order-5 FP64 kernel with gather warps, csf_column.cuh col_gather_role)
int enqueue_column(csf_ctx* c, const void* src, long long ld, void* dst, long long ld_dst, int nvec, double sc, int rot, double shift,
                   double* dCt, bool f32, const FusedGather* fg) {
    const int kind = column_kind(c); const bool ws = kind == 2;
    {
        const ColInfo ci = fg ? column_info_wide_p5_g() : column_info(c->p, kind);
        if (ci.smem > c->smem_optin) return fail(c, CSF_EUNSUPPORTED, "column tile does not fit shared memory");
        if (4 * ld >= (1LL << 31) || 4 * ld_dst >= (1LL << 31)) return fail(c, CSF_EUNSUPPORTED, "leading dimension too large");
        const int vpc = ci.lanes / 4;               // spinor vectors per CTA
        ColParams q{};
        const int n = c->n;
        const double hx2 = c->h[0] * c->h[0];
        for (int i = 0; i < n; ++i) {
            for (int j = 0; j < n; ++j) { q.Ah[i][j] = c->dir[0].A[i][j] * (0.5 * hx2); q.Ahf[i][j] = (float)q.Ah[i][j]; }
            q.uh[i] = c->dir[0].u[i]; q.uhf[i] = (float)q.uh[i];
        }
        q.ax = 2.0 / hx2; q.rho_y = hx2 / (c->h[1] * c->h[1]); q.rho_z = hx2 / (c->h[2] * c->h[2]);
        q.src = src; q.dst = dst; q.rs = (int)(4 * ld); q.rd = (int)(4 * ld_dst); q.nvec = nvec;
        {
            const cuuint64_t nfx = c->nfree[0], nfy = c->nfree[1], nfz = c->nfree[2], p = c->p;
            const cuuint64_t sd[4] = {(cuuint64_t)2 * nvec, 2 * nfx, nfy, nfz};
            const cuuint64_t rb = (cuuint64_t)ld * (f32 ? 8 : 16);        // bytes per spinor row
            if (rb % 16 != 0) return fail(c, CSF_EINVAL, "leading dimension of a complex64 block must be even");
            const cuuint64_t ss[3] = {rb, 2 * nfx * rb, nfy * 2 * nfx * rb};
            const cuuint32_t sb[4] = {(cuuint32_t)(ci.lanes / 2), (cuuint32_t)(2 * p), (cuuint32_t)p, (cuuint32_t)p};
            const cuuint64_t vd[3] = {4 * nfx, nfy, nfz};
            const cuuint64_t vs[2] = {nfx * 32, nfy * nfx * 32};
            const cuuint32_t vbx[3] = {(cuuint32_t)(4 * p), (cuuint32_t)p, (cuuint32_t)p};
            if (((uintptr_t)src & 15) != 0) return fail(c, CSF_EINVAL, "block pointer must be 16-byte aligned");
            if (!encode_map(&q.tm_src, src, 4, sd, ss, sb, f32) || !encode_map(&q.tm_vb, c->d_vb.p, 3, vd, vs, vbx))
                return fail(c, CSF_ECUDA, "cuTensorMapEncodeTiled failed");
        }
        q.ncx = c->ncell[0]; q.ncy = c->ncell[1]; q.ncz = c->ncell[2];
        q.nfx = c->nfree[0]; q.nfy = c->nfree[1]; q.nfz = c->nfree[2];
        q.bcx = c->bc[0]; q.bcy = c->bc[1]; q.bcz = c->bc[2];
        q.col_order = c->d_col_order.as<int>(); q.ncols = c->ncell[0] * c->ncell[1];
        // cells per z-segment: the warp-specialised kernel streams whole columns (up to 64 cells) through one CTA
        q.seg_len = std::min(c->seg_len > 0 ? c->seg_len : (ws ? 64 : 16), c->ncell[2]); q.nseg = (c->ncell[2] + q.seg_len - 1) / q.seg_len;
        q.nchunks = (nvec + vpc - 1) / vpc; q.chunk_group = std::min(c->chunk_group, q.nchunks);
        q.vb = c->d_vb.as<double>(); q.shift = shift; q.sc = sc; q.rot = rot & 3;
#ifdef WS_PROF
        {   // cycle counters of the last launch: [CTA][12 warps][4], dumped to CSF_WS_PROF_FILE by the previous launch's data
            static long long* dprof = nullptr; static std::vector<long long> hprof(148 * 12 * 4);
            if (!dprof) cudaMalloc(&dprof, hprof.size() * 8);
            else if (const char* f = std::getenv("CSF_WS_PROF_FILE")) {
                cudaStreamSynchronize(c->stream); cudaMemcpy(hprof.data(), dprof, hprof.size() * 8, cudaMemcpyDeviceToHost);
                if (FILE* fp = std::fopen(f, "w")) { for (size_t i = 0; i < hprof.size(); i += 4) std::fprintf(fp, "%lld %lld %lld %lld\n", hprof[i], hprof[i + 1], hprof[i + 2], hprof[i + 3]); std::fclose(fp); }
            }
            cudaMemsetAsync(dprof, 0, hprof.size() * 8, c->stream);
            q.prof = dprof;
        }
#endif
        const int kmode = column_mode(c, nvec, vpc, f32);
        const int lv = aux_warps(c, f32, kmode, kind) - 2;      // which sub-pair lists match the kernel's expansion-warp count
        if (c->natoms > 0) {
            q.sub_ptr = c->d_sub_ptr[lv].as<int>(); q.sub_desc = c->d_sub_desc[lv].as<int4>();
            q.ent_loc = c->d_ent_locf.as<int>();
            q.Ct = dCt; q.npjp = c->npjp; q.a_pack = c->d_a_pack[lv].as<double>();
        }
        const long long ngroups = (q.nchunks + q.chunk_group - 1) / q.chunk_group;
        long long nblocks = (long long)q.chunk_group * q.ncols * q.nseg * ngroups;
        if (nblocks > 0x7fffffffLL || (long long)q.nchunks * q.ncols * q.nseg > 0x7fffffffLL) return fail(c, CSF_EUNSUPPORTED, "grid too large");
        if (ws) nblocks = std::min<long long>((long long)q.nchunks * q.ncols * q.nseg, c->sm_count);      // persistent CTAs, one per SM
        if (fg) {
            // the gather warps' task list: (gather block, chunk of kCgVec vectors) of the OTHER block; its C is cleared here
            ColGather& g = q.g;
            g.src = static_cast<const double*>(fg->src); g.ld = fg->ld; g.nvec = fg->nvec;
            g.gb_atom = c->d_gb_atom.as<int>(); g.gb_beg = c->d_gb_beg.as<int>(); g.gb_end = c->d_gb_end.as<int>(); g.gb_k0 = c->d_gb_k0.as<int>();
            g.ent_node = c->d_ent_node.as<int>(); g.g_pack = c->d_g_pack.as<double>();
            g.atom_coff = c->d_atom_coff.as<long long>(); g.atom_npj = c->d_atom_npj.as<int>();
            g.C = fg->dC; g.ldc = fg->nvec;
            g.nvc = (fg->nvec + kCgVec - 1) / kCgVec; g.ntasks = fg->dC ? c->n_gather_blocks * g.nvc : 0;
            if (g.ntasks > 0) CSF_CUDA(c, cudaMemsetAsync(fg->dC, 0, (size_t)c->crows * g.ldc * sizeof(double2), c->stream));
        }
        {
            ProfScope ps(c, CSF_KIND_CELL);
            if (fg) CSF_CUDA(c, launch_column_wide_p5_g(c->npjp / 4, kmode, f32, q, nblocks, c->stream));
            else CSF_CUDA(c, launch_column(c->p, c->natoms > 0 ? c->npjp / 4 : 5, kmode, f32, kind, q, nblocks, c->stream));
        }
        c->launches += 1;
        return CSF_OK;
    }
}

// one step: dst += sc * i^rot * (Hhat - shift) src
// src, dst: complex128 blocks, or complex64 blocks when f32 (CSF_FP32_INTERMEDIATE)
int enqueue_step(csf_ctx* c, const void* src, long long ld, void* dst, long long ld_dst, int nvec, double sc, int rot, double shift,
                 double* dC, double* dCt, bool f32 = false) {
    // the sum-factorised kernels hold the Gamma-point operator with real projectors only
    if (c->kpt_on || c->proj_complex) return fail(c, CSF_ESTATE, "a k-point / complex projectors are set: only the dense path (csf_apply_H_dense, csf_filter_dense) serves them");
    if (c->natoms > 0) {
        int rc = enqueue_gather(c, src, ld, nvec, dC, f32); if (rc != CSF_OK) return rc;
        rc = enqueue_delta(c, dC, dCt, nvec, sc); if (rc != CSF_OK) return rc;
    }
    return enqueue_column(c, src, ld, dst, ld_dst, nvec, sc, rot, shift, dCt, f32, nullptr);
}

// The fused path of csf_filter (complex128, order 5, 8 vectors per CTA, 18 projectors per atom): the block is split into two
// halves whose column steps alternate, and each column launch computes, in two extra warps, the projector coefficients the
// OTHER half needs next. CSF_FUSED_GATHER=0 switches it off, =1 takes it for any block of >= 9 vectors (tests).
bool fused_gather_ok(const csf_ctx* c, int nvec) {
    if (c->fused_gather == 0 || column_kind(c) != 1 || c->p != 5 || c->natoms == 0 || c->npj_uniform != 18 || c->npjp != 20) return false;
    if (column_info_wide_p5_g().smem > c->smem_optin) return false;
    // (from 9 vectors on the first half is a multiple of 8 vectors, which keeps the two halves' C~ blocks inside ctp_bytes(nvec))
    if (c->fused_gather == 1) return nvec >= 9;
    // policy: both halves whole gather tasks of 32 vectors (a block of 96 = 48 + 48 pads the gather warps' work by a third and
    // measured 761 against 711 ms at config 3; 64 = 32 + 32 breaks even, 256 = 128 + 128 gains 3-7 %)
    return nvec >= 64 && nvec % 64 == 0;
}

size_t f32_block_bytes(const csf_ctx* c, int nvec) { return ((size_t)2 * c->M * ((nvec + 1) & ~1) * sizeof(float2) + 255) / 256 * 256; }
size_t block_bytes(const csf_ctx* c, int nvec) { return (size_t)2 * c->M * nvec * sizeof(double2); }
// C~ in fragment order: [atom][chunk][KS][L/8][32] doubles
size_t ctp_bytes(const csf_ctx* c, int nvec) {
    size_t best = 0;                           // the larger of the two lane counts the column kernel may run with
    for (int w = 0; w < 2; ++w) {
        const int lanes = column_info(c->p, w != 0).lanes, nchunks = (nvec + lanes / 4 - 1) / (lanes / 4);
        best = std::max(best, (size_t)c->natoms * nchunks * (c->npjp / 4) * (lanes / 8) * 32 * sizeof(double));
    }
    return (best + 255) / 256 * 256;
}
size_t coef_bytes(const csf_ctx* c, int nvec) { return ((size_t)c->crows * nvec * sizeof(double2) + 255) / 256 * 256; }

int enqueue_zero(csf_ctx* c, double* dst, long long ld, int nvec) {
    const long long rows = 2 * c->M;
    if (ld == nvec) { CSF_CUDA(c, cudaMemsetAsync(dst, 0, (size_t)rows * ld * sizeof(double2), c->stream)); return CSF_OK; }
    { ProfScope ps(c, CSF_KIND_AUX); zero_kernel<<<c->sm_count * 8, 256, 0, c->stream>>>(reinterpret_cast<double2*>(dst), rows, ld, nvec); }
    CSF_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return CSF_OK;
}

int check_block_args(csf_ctx* c, const void* x, const void* y, long long ld, int nvec, const void* work, size_t work_bytes, size_t need) {
    if (!c) return CSF_EINVAL;
    if (!x || !y) return fail(c, CSF_EINVAL, "NULL block pointer");
    if (x == y) return fail(c, CSF_EINVAL, "Y must not alias X");
    if (nvec < 0 || ld < nvec) return fail(c, CSF_EINVAL, "need 0 <= nvec <= ld");
    if (!c->have_pot && !(c->kpt_on || c->proj_complex)) return fail(c, CSF_ESTATE, "csf_set_potential has not been called");
    if (nvec > 0 && need > 0 && (!work || work_bytes < need)) return fail(c, CSF_EINVAL, "workspace too small");
    return CSF_OK;
}

}  // namespace

extern "C" {

const char* csf_last_error(const csf_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

int csf_create(csf_ctx** out, const int ncell[3], const double box[3], int order, const int bc[3], int device, void* cuda_stream) {
    CSF_GUARD_BEGIN
    if (!out || !ncell || !box || !bc) return fail(nullptr, CSF_EINVAL, "NULL argument");
    *out = nullptr;
    if (order < 1) return fail(nullptr, CSF_EINVAL, "order must be >= 1");
    if (order > 7) return fail(nullptr, CSF_EUNSUPPORTED, "order > 7 is not supported");
    long long M = 1, E = 1;
    for (int d = 0; d < 3; ++d) {
        if (ncell[d] < 1 || !(box[d] > 0.0)) return fail(nullptr, CSF_EINVAL, "ncell must be >= 1 and box > 0");
        if (bc[d] == CSF_BC_FREE) return fail(nullptr, CSF_EUNSUPPORTED, "CSF_BC_FREE is not supported on the GPU path");
        if (bc[d] != CSF_BC_PERIODIC && bc[d] != CSF_BC_DIRICHLET) return fail(nullptr, CSF_EINVAL, "bad boundary condition");
        long long nf = (long long)ncell[d] * order - (bc[d] == CSF_BC_DIRICHLET ? 1 : 0);
        if (nf < 1) return fail(nullptr, CSF_EINVAL, "direction has no unconstrained node");
        M *= nf; E *= ncell[d];
    }
    if (M >= (1LL << 31) || E >= (1LL << 31)) return fail(nullptr, CSF_EUNSUPPORTED, "mesh too large for 32-bit node ids");
    int ndev = 0;
    cudaError_t ce = cudaGetDeviceCount(&ndev);
    if (ce != cudaSuccess || ndev <= 0) return fail(nullptr, CSF_ECUDA, std::string("no CUDA device: ") + cudaGetErrorString(ce));
    if (device < 0 || device >= ndev) return fail(nullptr, CSF_EINVAL, "bad device ordinal");
    ce = cudaSetDevice(device);
    if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "cudaSetDevice");
    csf_ctx* c = new (std::nothrow) csf_ctx();
    if (!c) return fail(nullptr, CSF_ENOMEM, "out of host memory");
    struct Owner { csf_ctx* p; ~Owner() { delete p; } } owner{c};        // released on success
    c->device = device; c->stream = static_cast<cudaStream_t>(cuda_stream);
    c->p = order; c->n = order + 1; c->M = M; c->E = (int)E;
    for (int d = 0; d < 3; ++d) {
        c->ncell[d] = ncell[d]; c->bc[d] = bc[d]; c->box[d] = box[d]; c->h[d] = box[d] / ncell[d];
        c->nfree[d] = ncell[d] * order - (bc[d] == CSF_BC_DIRICHLET ? 1 : 0);
    }
    build_gll(order, &c->gll);
    for (int d = 0; d < 3; ++d) build_dir(c->gll, c->h[d], &c->dir[d]);
    cudaDeviceProp prop;
    ce = cudaGetDeviceProperties(&prop, device);
    if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "cudaGetDeviceProperties");
    c->sm_count = prop.multiProcessorCount; c->smem_optin = prop.sharedMemPerBlockOptin;
    // CSF_LANES pins the column kernel variant for the parity tests (both variants against the oracle on every case)
    if (const char* e = std::getenv("CSF_LANES")) { int v = std::atoi(e); if (v == 16 || v == 32) c->lanes_force = v; }
    if (const char* e = std::getenv("CSF_GATHER")) c->bulk_gather = std::strcmp(e, "reg") != 0;
    if (const char* e = std::getenv("CSF_FUSED_GATHER")) c->fused_gather = std::atoi(e) != 0 ? 1 : 0;
    if (const char* e = std::getenv("CSF_KERNEL")) c->kernel_force = std::strcmp(e, "ws") == 0 ? 2 : (std::strcmp(e, "wide") == 0 ? 1 : 0);
    const int B = 8;
    // traversal order of the (cx, cy) columns: 8x8 tiles, x fastest inside (neighbouring columns run together, so the
    // x / y faces they share are combined in L2)
    std::vector<int> col_v; col_v.reserve((size_t)ncell[0] * ncell[1]);
    for (int by = 0; by < ncell[1]; by += B) for (int bx = 0; bx < ncell[0]; bx += B)
        for (int y = by; y < std::min(by + B, ncell[1]); ++y) for (int x = bx; x < std::min(bx + B, ncell[0]); ++x) col_v.push_back(x + ncell[0] * y);
    ce = c->d_col_order.upload(col_v);
    if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "upload column order");
    owner.p = nullptr;
    *out = c;
    return CSF_OK;
    CSF_GUARD_END((csf_ctx*)nullptr)
}

int csf_destroy(csf_ctx* ctx) {
    if (!ctx) return CSF_OK;
    cudaSetDevice(ctx->device);
    delete ctx;
    return CSF_OK;
}

int csf_set_stream(csf_ctx* ctx, void* cuda_stream) { if (!ctx) return CSF_EINVAL; ctx->stream = static_cast<cudaStream_t>(cuda_stream); return CSF_OK; }

int csf_num_nodes(const csf_ctx* ctx, int64_t* M) { if (!ctx || !M) return CSF_EINVAL; *M = ctx->M; return CSF_OK; }

// 1-D axis data of direction d: coordinate and lumped mass of every unconstrained node
static void axis_tables(const csf_ctx* c, int d, std::vector<double>* x, std::vector<double>* m) {
    const int p = c->p, nf = c->nfree[d];
    x->assign(nf, 0.0); m->assign(nf, 0.0);
    for (int cell = 0; cell < c->ncell[d]; ++cell)
        for (int i = 0; i <= p; ++i) {
            const int f = cell * p + i; int g;
            if (c->bc[d] == CSF_BC_PERIODIC) g = f % (c->ncell[d] * p);
            else { if (f == 0 || f == c->ncell[d] * p) continue; g = f - 1; }
            (*m)[g] += 0.5 * c->h[d] * c->gll.w[i];
            if (!(c->bc[d] == CSF_BC_PERIODIC && cell == c->ncell[d] - 1 && i == p)) (*x)[g] = (cell + 0.5 * (c->gll.xi[i] + 1.0)) * c->h[d];
        }
}

int csf_node_coords(const csf_ctx* ctx, double* xyz) {
    CSF_GUARD_BEGIN
    if (!ctx || !xyz) return CSF_EINVAL;
    std::vector<double> ax[3], am[3];
    for (int d = 0; d < 3; ++d) axis_tables(ctx, d, &ax[d], &am[d]);
    long long I = 0;
    for (int z = 0; z < ctx->nfree[2]; ++z) for (int y = 0; y < ctx->nfree[1]; ++y) for (int x = 0; x < ctx->nfree[0]; ++x, ++I) {
        xyz[3 * I] = ax[0][x]; xyz[3 * I + 1] = ax[1][y]; xyz[3 * I + 2] = ax[2][z];
    }
    return CSF_OK;
    CSF_GUARD_END(ctx)
}

int csf_mass_diag(const csf_ctx* ctx, double* mh) {
    CSF_GUARD_BEGIN
    if (!ctx || !mh) return CSF_EINVAL;
    std::vector<double> ax[3], am[3];
    for (int d = 0; d < 3; ++d) axis_tables(ctx, d, &ax[d], &am[d]);
    long long I = 0;
    for (int z = 0; z < ctx->nfree[2]; ++z) for (int y = 0; y < ctx->nfree[1]; ++y) for (int x = 0; x < ctx->nfree[0]; ++x, ++I)
        mh[I] = am[0][x] * am[1][y] * am[2][z];
    return CSF_OK;
    CSF_GUARD_END(ctx)
}

int csf_set_potential(csf_ctx* c, const double* veff, const double* bxyz) {
    CSF_GUARD_BEGIN
    if (!c) return CSF_EINVAL;
    if (!veff) return fail(c, CSF_EINVAL, "veff is NULL");
    CSF_CUDA(c, cudaSetDevice(c->device));
    std::vector<double> vb((size_t)c->M * 4);
    for (long long I = 0; I < c->M; ++I) {
        vb[4 * I] = veff[I];
        vb[4 * I + 1] = bxyz ? bxyz[3 * I] : 0.0; vb[4 * I + 2] = bxyz ? bxyz[3 * I + 1] : 0.0; vb[4 * I + 3] = bxyz ? bxyz[3 * I + 2] : 0.0;
    }
    CSF_CUDA(c, cudaStreamSynchronize(c->stream));
    CSF_CUDA(c, c->d_vb.upload(vb));
    c->have_pot = true;
    return CSF_OK;
    CSF_GUARD_END(c)
}

// pvals_im: NULL, or the imaginary parts of complex projector entries (csf_set_projectors_complex; same layout as pvals)
static int set_projectors_impl(csf_ctx* c, int natoms, const int64_t* node_ptr, const int64_t* node_idx, const int* nproj,
                               const double* pvals, const double* pvals_im, const int* atom_type, int ntypes, const csf_c128* delta, const int64_t* delta_ptr) {
    CSF_GUARD_BEGIN
    if (!c) return CSF_EINVAL;
    if (natoms < 0) return fail(c, CSF_EINVAL, "natoms < 0");
    CSF_CUDA(c, cudaSetDevice(c->device));
    CSF_CUDA(c, cudaStreamSynchronize(c->stream));
    c->natoms = 0; c->crows = 0; c->n_gather_blocks = 0; c->proj_complex = false;
    if (natoms == 0) return CSF_OK;
    if (!node_ptr || !node_idx || !nproj || !pvals || !atom_type || ntypes < 1 || !delta || !delta_ptr) return fail(c, CSF_EINVAL, "NULL projector argument");
    int npj_max = 0; bool uniform = true;
    for (int a = 0; a < natoms; ++a) {
        if (nproj[a] < 1) return fail(c, CSF_EINVAL, "nproj must be >= 1");
        if (atom_type[a] < 0 || atom_type[a] >= ntypes) return fail(c, CSF_EINVAL, "atom_type out of range");
        if (delta_ptr[atom_type[a] + 1] - delta_ptr[atom_type[a]] != (int64_t)4 * nproj[a] * nproj[a]) return fail(c, CSF_EINVAL, "Delta size does not match nproj");
        if (node_ptr[a + 1] < node_ptr[a]) return fail(c, CSF_EINVAL, "node_ptr not monotone");
        npj_max = std::max(npj_max, nproj[a]); uniform = uniform && nproj[a] == nproj[0];
    }
    if (npj_max > 32) return fail(c, CSF_EUNSUPPORTED, "more than 32 projectors per atom");
    const long long nent = node_ptr[natoms];
    if (nent >= (1LL << 31)) return fail(c, CSF_EUNSUPPORTED, "too many projector entries");
    for (long long t = 0; t < nent; ++t) if (node_idx[t] < 0 || node_idx[t] >= c->M) return fail(c, CSF_EINVAL, "node_idx out of range");
    const int p = c->p, npjp = npj_max <= 20 ? 20 : 32;   // whole DMMA k-steps of 4 projectors
    std::vector<double> mass((size_t)c->M);
    csf_mass_diag(c, mass.data());
    // owner cell and local index of every support node; sort each atom's entries by (cell, lz, ly, lx)
    struct Ent { int cell, lz, ly, lx; long long t; };
    std::vector<int> ent_node((size_t)nent), ent_locf((size_t)nent);
    std::vector<double> ent_p((size_t)nent * npjp, 0.0), ent_pi(pvals_im ? (size_t)nent * npjp : 0, 0.0);
    std::vector<long long> atom_coff(natoms); std::vector<int> atom_npj(nproj, nproj + natoms), atom_ty(atom_type, atom_type + natoms);
    std::vector<int> gb_atom, gb_beg, gb_end;
    struct Pair { int cell, atom; int off[kTabN + 1]; };
    std::vector<Pair> pairs;
    long long pv_off = 0, crows = 0;
    std::vector<Ent> ents;
    for (int a = 0; a < natoms; ++a) {
        atom_coff[a] = crows; crows += 2 * nproj[a];
        const long long t0 = node_ptr[a], t1 = node_ptr[a + 1];
        ents.clear(); ents.reserve(t1 - t0);
        for (long long t = t0; t < t1; ++t) {
            long long I = node_idx[t]; int g[3] = { (int)(I % c->nfree[0]), (int)((I / c->nfree[0]) % c->nfree[1]), (int)(I / ((long long)c->nfree[0] * c->nfree[1])) };
            int cl[3], lo[3];
            for (int d = 0; d < 3; ++d) { int f = g[d] + (c->bc[d] == CSF_BC_DIRICHLET ? 1 : 0); cl[d] = f / p; lo[d] = f % p; }
            ents.push_back({ cl[0] + c->ncell[0] * (cl[1] + c->ncell[1] * cl[2]), lo[2], lo[1], lo[0], t });
        }
        std::sort(ents.begin(), ents.end(), [](const Ent& x, const Ent& y) {
            if (x.cell != y.cell) return x.cell < y.cell; if (x.lz != y.lz) return x.lz < y.lz; if (x.ly != y.ly) return x.ly < y.ly; return x.lx < y.lx; });
        for (size_t q = 1; q < ents.size(); ++q)
            if (ents[q].cell == ents[q - 1].cell && ents[q].lz == ents[q - 1].lz && ents[q].ly == ents[q - 1].ly && ents[q].lx == ents[q - 1].lx)
                return fail(c, CSF_EINVAL, "duplicate node in an atom's support");
        for (size_t q = 0; q < ents.size(); ++q) {
            const long long e = t0 + (long long)q, t = ents[q].t, I = node_idx[t];
            ent_node[e] = (int)I; ent_locf[e] = (ents[q].lz * p + ents[q].ly) * p + ents[q].lx;
            const double s = 1.0 / std::sqrt(mass[I]);
            for (int x = 0; x < nproj[a]; ++x) ent_p[(size_t)e * npjp + x] = s * pvals[pv_off + (t - t0) * nproj[a] + x];
            if (pvals_im) for (int x = 0; x < nproj[a]; ++x) ent_pi[(size_t)e * npjp + x] = s * pvals_im[pv_off + (t - t0) * nproj[a] + x];
            if (q == 0 || ents[q].cell != ents[q - 1].cell) {
                Pair pr; pr.cell = ents[q].cell; pr.atom = a;
                for (int k = 0; k <= p; ++k) pr.off[k] = (int)e;
                pairs.push_back(pr);
            }
            Pair& pr = pairs.back();
            for (int k = ents[q].lz + 1; k <= p; ++k) pr.off[k] = (int)e + 1;
        }
        for (long long b = t0; b < t1; b += 256) { gb_atom.push_back(a); gb_beg.push_back((int)b); gb_end.push_back((int)std::min(b + 256, t1)); }
        pv_off += (t1 - t0) * nproj[a];
    }
    // P~^T of every k-step (4 entries, aligned to the atom's first entry) in DMMA A-fragment order for the gather kernel:
    // [k-step][m-tile][lane = (chi % 8) * 4 + entry % 4]
    const int mt = npjp <= 24 ? 3 : 4;
    std::vector<int> gb_k0(gb_atom.size());
    std::vector<long long> atom_k0(natoms + 1, 0);
    for (int a = 0; a < natoms; ++a) atom_k0[a + 1] = atom_k0[a] + (node_ptr[a + 1] - node_ptr[a] + 3) / 4;
    if (atom_k0[natoms] >= (1LL << 31)) return fail(c, CSF_EUNSUPPORTED, "too many projector entries");
    for (size_t b = 0; b < gb_atom.size(); ++b) gb_k0[b] = (int)(atom_k0[gb_atom[b]] + (gb_beg[b] - node_ptr[gb_atom[b]]) / 4);
    std::vector<double> g_pack((size_t)atom_k0[natoms] * mt * 32, 0.0);
    for (int a = 0; a < natoms; ++a)
        for (long long e = node_ptr[a]; e < node_ptr[a + 1]; ++e) {
            const size_t kstep = (size_t)atom_k0[a] + (e - node_ptr[a]) / 4; const int kq = (int)((e - node_ptr[a]) % 4);
            for (int x = 0; x < nproj[a]; ++x) g_pack[(kstep * mt + x / 8) * 32 + (x % 8) * 4 + kq] = ent_p[(size_t)e * npjp + x];
        }
    if (pvals_im) {                             // Im P~ in the same order (dense path only)
        std::vector<double> g_pack_im(g_pack.size(), 0.0);
        for (int a = 0; a < natoms; ++a)
            for (long long e = node_ptr[a]; e < node_ptr[a + 1]; ++e) {
                const size_t kstep = (size_t)atom_k0[a] + (e - node_ptr[a]) / 4; const int kq = (int)((e - node_ptr[a]) % 4);
                for (int x = 0; x < nproj[a]; ++x) g_pack_im[(kstep * mt + x / 8) * 32 + (x % 8) * 4 + kq] = ent_pi[(size_t)e * npjp + x];
            }
        CSF_CUDA(c, c->d_g_pack_im.upload(g_pack_im));
    }
    // sub-pairs for the column kernels: every (cell, atom) pair split into the owned-node row ranges of the nq expansion
    // warps (entries of a pair are sorted by that index), grouped by (cell, warp)
    if (crows >= (1LL << 31)) return fail(c, CSF_EUNSUPPORTED, "too many projector rows");
    for (int lv = 0; lv < kColMaxAuxWarps - 1; ++lv) {
    const int nq = 2 + lv;
    bool used = false;                          // does any kernel this context can run have nq expansion warps?
    for (int f = 0; f < 2; ++f) for (int md = 0; md < 3; ++md) used = used || aux_warps(c, f != 0, md, column_kind(c)) == nq;
    if (!used) continue;
    struct Sub { int key; int4 d; };
    std::vector<Sub> subs; subs.reserve(nq * pairs.size());
    for (const Pair& pr : pairs) {
        const int e1 = pr.off[p];
        int e = pr.off[0];
        for (int r = 0; r < nq; ++r) {
            int em = e; while (em < e1 && ent_locf[em] < col_aux_row0(p * p * p, nq, r + 1)) ++em;
            if (em > e) subs.push_back({pr.cell * nq + r, make_int4(pr.atom, 0, e, em)});
            e = em;
        }
    }
    std::stable_sort(subs.begin(), subs.end(), [](const Sub& x, const Sub& y) { return x.key < y.key; });
    std::vector<int> sub_ptr(nq * (size_t)c->E + 1, 0); std::vector<int4> sub_desc(subs.size());
    long long ntiles = 0;
    for (size_t q = 0; q < subs.size(); ++q) {
        sub_ptr[subs[q].key + 1]++;
        subs[q].d.y = (int)ntiles; ntiles += (subs[q].d.w - subs[q].d.z + 7) / 8;
        sub_desc[q] = subs[q].d;
    }
    if (ntiles >= (1LL << 31)) return fail(c, CSF_EUNSUPPORTED, "too many projector tiles");
    for (size_t q = 0; q < nq * (size_t)c->E; ++q) sub_ptr[q + 1] += sub_ptr[q];
    // P~ of every tile (8 rows of a sub-pair) in the order of the DMMA A fragment: [tile][k-step][lane = row*4 + k]
    const int ks = npjp / 4;
    std::vector<double> a_pack((size_t)ntiles * ks * 32, 0.0);
    for (const Sub& sb : subs)
        for (int e = sb.d.z; e < sb.d.w; ++e) {
            const size_t tile = (size_t)sb.d.y + (e - sb.d.z) / 8; const int row = (e - sb.d.z) % 8;
            for (int x = 0; x < npjp; ++x) a_pack[(tile * ks + x / 4) * 32 + row * 4 + x % 4] = ent_p[(size_t)e * npjp + x];
        }
    CSF_CUDA(c, c->d_sub_ptr[lv].upload(sub_ptr)); CSF_CUDA(c, c->d_sub_desc[lv].upload(sub_desc)); CSF_CUDA(c, c->d_a_pack[lv].upload(a_pack));
    }
    std::vector<double2> dl((size_t)delta_ptr[ntypes]);
    for (size_t i = 0; i < dl.size(); ++i) dl[i] = make_double2(delta[i].re, delta[i].im);
    std::vector<long long> dptr(delta_ptr, delta_ptr + ntypes + 1);
    CSF_CUDA(c, c->d_ent_locf.upload(ent_locf)); CSF_CUDA(c, c->d_ent_node.upload(ent_node));
    CSF_CUDA(c, c->d_atom_coff.upload(atom_coff)); CSF_CUDA(c, c->d_atom_npj.upload(atom_npj)); CSF_CUDA(c, c->d_atom_type.upload(atom_ty));
    CSF_CUDA(c, c->d_delta.upload(dl)); CSF_CUDA(c, c->d_delta_ptr.upload(dptr));
    CSF_CUDA(c, c->d_gb_k0.upload(gb_k0)); CSF_CUDA(c, c->d_g_pack.upload(g_pack)); CSF_CUDA(c, c->d_gb_atom.upload(gb_atom)); CSF_CUDA(c, c->d_gb_beg.upload(gb_beg)); CSF_CUDA(c, c->d_gb_end.upload(gb_end));
    c->natoms = natoms; c->crows = crows; c->npjp = npjp; c->npj_uniform = uniform ? nproj[0] : 0;
    c->n_gather_blocks = (int)gb_atom.size();
    c->proj_complex = pvals_im != nullptr;
    return CSF_OK;
    CSF_GUARD_END(c)
}

int csf_set_projectors(csf_ctx* c, int natoms, const int64_t* node_ptr, const int64_t* node_idx, const int* nproj,
                       const double* pvals, const int* atom_type, int ntypes, const csf_c128* delta, const int64_t* delta_ptr) {
    return set_projectors_impl(c, natoms, node_ptr, node_idx, nproj, pvals, nullptr, atom_type, ntypes, delta, delta_ptr);
}

int csf_set_projectors_complex(csf_ctx* c, int natoms, const int64_t* node_ptr, const int64_t* node_idx, const int* nproj,
                               const csf_c128* pvals, const int* atom_type, int ntypes, const csf_c128* delta, const int64_t* delta_ptr) {
    CSF_GUARD_BEGIN
    if (!c) return CSF_EINVAL;
    if (natoms <= 0 || !node_ptr || !nproj || !pvals) return set_projectors_impl(c, natoms, node_ptr, node_idx, nproj, nullptr, nullptr, atom_type, ntypes, delta, delta_ptr);
    for (int a = 0; a < natoms; ++a) if (nproj[a] < 1 || node_ptr[a + 1] < node_ptr[a]) return fail(c, CSF_EINVAL, "bad nproj / node_ptr");
    size_t n = 0;
    for (int a = 0; a < natoms; ++a) n += (size_t)(node_ptr[a + 1] - node_ptr[a]) * nproj[a];
    std::vector<double> re(n), im(n);
    for (size_t i = 0; i < n; ++i) { re[i] = pvals[i].re; im[i] = pvals[i].im; }
    return set_projectors_impl(c, natoms, node_ptr, node_idx, nproj, re.data(), im.data(), atom_type, ntypes, delta, delta_ptr);
    CSF_GUARD_END(c)
}

int csf_workspace_bytes(const csf_ctx* c, int nvec, int mode, size_t* bytes) {
    if (!c || !bytes || nvec < 0) return CSF_EINVAL;
    if (mode == CSF_FP32_INTERMEDIATE) {
        // two complex64 blocks with an even leading dimension (16-byte rows for TMA) = the bytes of one complex128 block
        *bytes = f32_block_bytes(c, nvec) * 2 + coef_bytes(c, nvec) + ctp_bytes(c, nvec) + 256;
        return CSF_OK;
    }
    if (mode != CSF_FP64) return CSF_EUNSUPPORTED;
    *bytes = block_bytes(c, nvec) + coef_bytes(c, nvec) + ctp_bytes(c, nvec) + 256;
    return CSF_OK;
}

int csf_apply_H(csf_ctx* c, const csf_c128* dX, csf_c128* dY, int64_t ld, int nvec, void* d_work, size_t work_bytes) {
    CSF_GUARD_BEGIN
    if (!c) return CSF_EINVAL;
    const size_t need = c->natoms > 0 ? coef_bytes(c, std::max(nvec, 0)) + ctp_bytes(c, std::max(nvec, 0)) : 0;
    int rc = check_block_args(c, dX, dY, ld, nvec, d_work, work_bytes, need);
    if (rc != CSF_OK || nvec == 0) return rc;
    CSF_CUDA(c, cudaSetDevice(c->device));
    double* dC = static_cast<double*>(d_work);
    double* dCt = reinterpret_cast<double*>(static_cast<char*>(d_work) + coef_bytes(c, nvec));
    rc = enqueue_zero(c, reinterpret_cast<double*>(dY), ld, nvec);
    if (rc != CSF_OK) return rc;
    return enqueue_step(c, reinterpret_cast<const double*>(dX), ld, reinterpret_cast<double*>(dY), ld, nvec, 1.0, 0, 0.0, dC, dCt);
    CSF_GUARD_END(c)
}

}  // extern "C"

// Scratch of csf_apply_H_static: part of the library image, resident on every GPU that loads it, never freed.
// In host code the name is only a handle for cudaGetSymbolAddress: it is NOT a device address and is never passed to a kernel.
static __device__ __align__(256) unsigned char g_static_scratch[CSF_STATIC_SCRATCH_BYTES];

namespace {
// device address of g_static_scratch on the context's device (which must be current), resolved once per device
int static_scratch_address(csf_ctx* c, unsigned char** out) {
    static unsigned char* addr[64] = {};
    static std::mutex mu;
    if (c->device < 0 || c->device >= 64) return fail(c, CSF_EUNSUPPORTED, "device ordinal >= 64");
    std::lock_guard<std::mutex> lk(mu);
    if (!addr[c->device]) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return cuda_fail(c, e, "cudaGetSymbolAddress(g_static_scratch)");
        if (!p || ((uintptr_t)p & 255) != 0) return fail(c, CSF_ECUDA, "static scratch has no usable device address");
        addr[c->device] = static_cast<unsigned char*>(p);
    }
    *out = addr[c->device];
    return CSF_OK;
}
}  // namespace

extern "C" {

int csf_apply_H_static(csf_ctx* c, const csf_c128* dX, csf_c128* dY, int64_t ld, int nvec) {
    CSF_GUARD_BEGIN
    if (!c) return CSF_EINVAL;
    int rc = check_block_args(c, dX, dY, ld, nvec, nullptr, 0, 0);
    if (rc != CSF_OK || nvec == 0) return rc;
    if (c->prof) return fail(c, CSF_ESTATE, "csf_apply_H_static: switch per-kernel profiling off first (it creates events)");
    const size_t cb = c->natoms > 0 ? coef_bytes(c, nvec) : 0, need = c->natoms > 0 ? cb + ctp_bytes(c, nvec) : 0;
    if (need > (size_t)CSF_STATIC_SCRATCH_BYTES)
        return fail(c, CSF_EUNSUPPORTED, "csf_apply_H_static: projector scratch of " + std::to_string(need) + " bytes for nvec = " + std::to_string(nvec) +
                    " exceeds the static limit of " + std::to_string((size_t)CSF_STATIC_SCRATCH_BYTES) + " bytes; use csf_apply_H with a workspace, or fewer vectors per call");
    CSF_CUDA(c, cudaSetDevice(c->device));
    unsigned char* scratch = nullptr;
    if (need > 0) { rc = static_scratch_address(c, &scratch); if (rc != CSF_OK) return rc; }
    // enqueue_step clears C and C~ on the stream before the gather / Delta kernels add into them
    double* dC = reinterpret_cast<double*>(scratch);
    double* dCt = reinterpret_cast<double*>(scratch + cb);
    rc = enqueue_zero(c, reinterpret_cast<double*>(dY), ld, nvec);
    if (rc != CSF_OK) return rc;
    return enqueue_step(c, reinterpret_cast<const double*>(dX), ld, reinterpret_cast<double*>(dY), ld, nvec, 1.0, 0, 0.0, dC, dCt);
    CSF_GUARD_END(c)
}

// the launch sequence of one filter call on c->stream (arguments already checked)
static int filter_enqueue(csf_ctx* c, const csf_c128* dX, csf_c128* dY, int64_t ld, int nvec, int degree, double a, double b, int mode, void* d_work) {
    int rc = CSF_OK;
    const long long rows = 2 * c->M;
    const double cc = 0.5 * (a + b), ee = 0.5 * (b - a);
    const double2* X = reinterpret_cast<const double2*>(dX);
    double* Y = reinterpret_cast<double*>(dY);
    if (degree == 0) {
        { ProfScope ps(c, CSF_KIND_AUX); rot_copy_kernel<<<c->sm_count * 8, 256, 0, c->stream>>>(X, ld, reinterpret_cast<double2*>(Y), ld, rows, nvec, 0); }
        CSF_CUDA(c, cudaGetLastError()); c->launches += 1;
        return CSF_OK;
    }
    char* w = static_cast<char*>(d_work);
    if (mode == CSF_FP32_INTERMEDIATE) {
        // The same recurrence with both block buffers in complex64 and FP32 cell arithmetic; X is narrowed on the way in
        // (W_0 = i^m X), W_m is widened into Y. Projector coefficients C, C~ stay in FP64.
        const long long ldw = (nvec + 1) & ~1;
        float2* f0 = reinterpret_cast<float2*>(w);
        float2* f1 = reinterpret_cast<float2*>(w + f32_block_bytes(c, nvec));
        double* fC = reinterpret_cast<double*>(w + 2 * f32_block_bytes(c, nvec));
        double* fCt = reinterpret_cast<double*>(w + 2 * f32_block_bytes(c, nvec) + coef_bytes(c, nvec));
        { ProfScope ps(c, CSF_KIND_AUX); rot_narrow_kernel<<<c->sm_count * 8, 256, 0, c->stream>>>(X, ld, f0, ldw, rows, nvec, degree & 3); }
        CSF_CUDA(c, cudaGetLastError()); c->launches += 1;
        CSF_CUDA(c, cudaMemsetAsync(f1, 0, (size_t)rows * ldw * sizeof(float2), c->stream));
        // W_1 = (-i/e)(Hhat - c) W_0, then W_{k+1} = W_{k-1} + (-2i/e)(Hhat - c) W_k
        for (int k = 0; k < degree; ++k) {
            const bool odd = (k & 1);
            rc = enqueue_step(c, odd ? f1 : f0, ldw, odd ? f0 : f1, ldw, nvec, (k == 0 ? 1.0 : 2.0) / ee, 3, cc, fC, fCt, true);
            if (rc != CSF_OK) return rc;
        }
        { ProfScope ps(c, CSF_KIND_AUX); widen_kernel<<<c->sm_count * 8, 256, 0, c->stream>>>((degree & 1) ? f1 : f0, ldw, reinterpret_cast<double2*>(Y), ld, rows, nvec); }
        CSF_CUDA(c, cudaGetLastError()); c->launches += 1;
        return CSF_OK;
    }
    double* Wk = reinterpret_cast<double*>(w);                              // the second block buffer, [2M][nvec]
    double* dC = reinterpret_cast<double*>(w + block_bytes(c, nvec));
    double* dCt = reinterpret_cast<double*>(w + block_bytes(c, nvec) + coef_bytes(c, nvec));
    // W_k = i^(m-k) T_k(H~) X, so that W_{k+1} = W_{k-1} + (-2i/e)(Hhat - c) W_k and W_m = T_m(H~) X.
    // W_0 lives in the buffer that also receives W_m: Y if m is even, the workspace block if m is odd.
    const bool even_m = (degree % 2 == 0);
    double* buf0 = even_m ? Y : Wk;  const long long ld0 = even_m ? ld : nvec;
    double* buf1 = even_m ? Wk : Y;  const long long ld1 = even_m ? nvec : ld;
    if (degree >= 2) {
        { ProfScope ps(c, CSF_KIND_AUX); rot_copy_kernel<<<c->sm_count * 8, 256, 0, c->stream>>>(X, ld, reinterpret_cast<double2*>(buf0), ld0, rows, nvec, degree & 3); }   // W_0 = i^m X
        CSF_CUDA(c, cudaGetLastError()); c->launches += 1;
    }
    rc = enqueue_zero(c, buf1, ld1, nvec); if (rc != CSF_OK) return rc;
    if (fused_gather_ok(c, nvec)) {
        // Two half-blocks (the first a multiple of 8 vectors), column steps alternating: K(h, k) = step k on half h. The gather
        // warps of K(0, k) compute C of (1, k), those of K(1, k) C of (0, k + 1): both sources are complete by then, because
        // the launches of one stream run in order. Only C of (0, 0) needs the gather kernel.
        if (c->kpt_on || c->proj_complex) return fail(c, CSF_ESTATE, "a k-point / complex projectors are set: only the dense path (csf_apply_H_dense, csf_filter_dense) serves them");
        const int nv0 = std::min(nvec - 1, ((nvec + 1) / 2 + 7) / 8 * 8), nvh[2] = {nv0, nvec - nv0}, voff[2] = {0, nv0};
        double* hC[2] = {dC, dC + (size_t)c->crows * nv0 * 2};
        double* hCt[2] = {dCt, reinterpret_cast<double*>(reinterpret_cast<char*>(dCt) + ctp_bytes(c, nv0))};
        auto src_of = [&](int h, int k, long long* lds) -> const double* {
            if (k == 0) { *lds = ld; return reinterpret_cast<const double*>(dX) + 2 * (size_t)voff[h]; }
            const bool odd = (k & 1);
            *lds = odd ? ld1 : ld0; return (odd ? buf1 : buf0) + 2 * (size_t)voff[h];
        };
        long long lds = 0;
        const double* s00 = src_of(0, 0, &lds);
        rc = enqueue_gather(c, s00, lds, nvh[0], hC[0], false); if (rc != CSF_OK) return rc;
        rc = enqueue_delta(c, hC[0], hCt[0], nvh[0], 1.0); if (rc != CSF_OK) return rc;
        for (int k = 0; k < degree; ++k) {
            const bool odd = (k & 1);
            double* dstb = (k == 0) ? buf1 : (odd ? buf0 : buf1); const long long ldd = (k == 0) ? ld1 : (odd ? ld0 : ld1);
            const double sc = (k == 0 ? 1.0 : 2.0) / ee; const int rot = (k == 0) ? ((degree + 3) & 3) : 3;
            for (int h = 0; h < 2; ++h) {
                const int hn = 1 - h, kn = (h == 0) ? k : k + 1;         // whose coefficients this launch gathers
                FusedGather fg{nullptr, 0, nvh[hn], nullptr};
                if (kn < degree) { long long ldn = 0; fg.src = src_of(hn, kn, &ldn); fg.ld = ldn; fg.dC = hC[hn]; }
                const double* srcp = src_of(h, k, &lds);
                rc = enqueue_column(c, srcp, lds, dstb + 2 * (size_t)voff[h], ldd, nvh[h], sc, rot, cc, hCt[h], false, &fg);
                if (rc != CSF_OK) return rc;
                if (kn < degree) { rc = enqueue_delta(c, hC[hn], hCt[hn], nvh[hn], 1.0, kn == 0); if (rc != CSF_OK) return rc; }
            }
        }
        return CSF_OK;
    }
    // W_1 = (i^(m-1)/e)(Hhat - c) X
    rc = enqueue_step(c, reinterpret_cast<const double*>(dX), ld, buf1, ld1, nvec, 1.0 / ee, (degree + 3) & 3, cc, dC, dCt);
    if (rc != CSF_OK) return rc;
    for (int k = 1; k < degree; ++k) {
        const bool odd = (k & 1);
        rc = enqueue_step(c, odd ? buf1 : buf0, odd ? ld1 : ld0, odd ? buf0 : buf1, odd ? ld0 : ld1, nvec, 2.0 / ee, 3, cc, dC, dCt);
        if (rc != CSF_OK) return rc;
    }
    return CSF_OK;
}

int csf_filter(csf_ctx* c, const csf_c128* dX, csf_c128* dY, int64_t ld, int nvec, int degree, double a, double b, int mode,
               void* d_work, size_t work_bytes) {
    CSF_GUARD_BEGIN
    if (!c) return CSF_EINVAL;
    if (mode != CSF_FP64 && mode != CSF_FP32_INTERMEDIATE) return fail(c, CSF_EINVAL, "unknown mode");
    if (degree < 0) return fail(c, CSF_EINVAL, "degree < 0");
    if (!(a < b)) return fail(c, CSF_EINVAL, "need a < b");
    size_t need = 0;
    if (nvec > 0) csf_workspace_bytes(c, nvec, mode, &need);
    int rc = check_block_args(c, dX, dY, ld, nvec, d_work, work_bytes, degree >= 1 ? need : 0);
    if (rc != CSF_OK || nvec == 0) return rc;
    CSF_CUDA(c, cudaSetDevice(c->device));
    // (Replaying the sequence as a CUDA graph was measured at config 1, the launch-bound one: 11.40 against 11.48 ms per block.
    // The gaps are on the device, not in the launch path; the graph was dropped.)
    return filter_enqueue(c, dX, dY, ld, nvec, degree, a, b, mode, d_work);
    CSF_GUARD_END(c)
}

int csf_filter_host(csf_ctx* c, const csf_c128* hX, csf_c128* hY, int64_t ld, int nvec, int degree, double a, double b, int mode) {
    CSF_GUARD_BEGIN
    if (!c) return CSF_EINVAL;
    if (!hX || !hY) return fail(c, CSF_EINVAL, "NULL host block pointer");
    if (nvec < 0 || ld < nvec) return fail(c, CSF_EINVAL, "need 0 <= nvec <= ld");
    if (degree < 0) return fail(c, CSF_EINVAL, "degree < 0");
    if (!(a < b)) return fail(c, CSF_EINVAL, "need a < b");
    if (!c->have_pot) return fail(c, CSF_ESTATE, "csf_set_potential has not been called");
    if (nvec == 0) return CSF_OK;
    CSF_CUDA(c, cudaSetDevice(c->device));
    const int chunk = std::min(c->host_chunk, nvec);
    // Column chunks. What the pipeline cannot hide is the host->device copy of the first chunk and the device->host copy of the
    // last one, so a block of at least three chunks starts and ends with half a chunk (a multiple of 8 columns). Not less:
    // narrow blocks filter slowly (config 3: 6.9 ms per column at 64 columns and more, 7.8 at 48, 11.5 at 16), and a quarter
    // chunk at both ends measured no gain at all.
    std::vector<int> csz;
    {
        const int q2 = chunk / 2 / 8 * 8;
        int mid = nvec;
        const bool ramp = nvec >= 3 * chunk && q2 >= 8;
        if (ramp) { csz.push_back(q2); mid -= 2 * q2; }
        for (; mid > 0; mid -= chunk) csz.push_back(std::min(chunk, mid));
        if (ramp) csz.push_back(q2);
    }
    const int nch = (int)csz.size();
    size_t wb = 0;
    int rc = csf_workspace_bytes(c, chunk, mode, &wb); if (rc != CSF_OK) return fail(c, rc, "unsupported mode");
    const size_t rows = (size_t)2 * c->M, cb = rows * chunk * sizeof(double2);
    for (int s = 0; s < (nch > 1 ? 2 : 1); ++s) {
        if (c->h_x[s].bytes < cb) CSF_CUDA(c, c->h_x[s].alloc(cb));
        if (c->h_y[s].bytes < cb) CSF_CUDA(c, c->h_y[s].alloc(cb));
    }
    if (c->h_w.bytes < wb) CSF_CUDA(c, c->h_w.alloc(wb));
    if (!c->hs_in) {
        CSF_CUDA(c, cudaStreamCreateWithFlags(&c->hs_in, cudaStreamNonBlocking));
        CSF_CUDA(c, cudaStreamCreateWithFlags(&c->hs_out, cudaStreamNonBlocking));
        for (int s = 0; s < 2; ++s) {
            CSF_CUDA(c, cudaEventCreateWithFlags(&c->ev_in[s], cudaEventDisableTiming));
            CSF_CUDA(c, cudaEventCreateWithFlags(&c->ev_cmp[s], cudaEventDisableTiming));
            CSF_CUDA(c, cudaEventCreateWithFlags(&c->ev_out[s], cudaEventDisableTiming));
        }
    }
    // chunk i: host->device on hs_in, filter on the context's stream, device->host on hs_out; slot i%2 is reused
    // only after chunk i-2 has been filtered (x slot) and copied out (y slot), so copies overlap the filter.
    // an error inside the pipeline must not return while copies into the caller's host memory are in flight
    auto drain = [&]() { cudaStreamSynchronize(c->hs_in); cudaStreamSynchronize(c->stream); cudaStreamSynchronize(c->hs_out); };
#define CSF_CUDA_H(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { drain(); return cuda_fail(c, e__, #call); } } while (0)
    int v0 = 0;
    for (int i = 0; i < nch; v0 += csz[i], ++i) {
        const int s = i & 1, nv = csz[i];
        const size_t wbytes = (size_t)nv * sizeof(double2);
        if (i >= 2) CSF_CUDA_H(cudaStreamWaitEvent(c->hs_in, c->ev_cmp[s], 0));
        CSF_CUDA_H(cudaMemcpy2DAsync(c->h_x[s].p, wbytes, hX + v0, (size_t)ld * sizeof(double2), wbytes, rows, cudaMemcpyHostToDevice, c->hs_in));
        CSF_CUDA_H(cudaEventRecord(c->ev_in[s], c->hs_in));
        CSF_CUDA_H(cudaStreamWaitEvent(c->stream, c->ev_in[s], 0));
        if (i >= 2) CSF_CUDA_H(cudaStreamWaitEvent(c->stream, c->ev_out[s], 0));
        rc = csf_filter(c, static_cast<const csf_c128*>(c->h_x[s].p), static_cast<csf_c128*>(c->h_y[s].p), nv, nv, degree, a, b, mode, c->h_w.p, c->h_w.bytes);
        if (rc != CSF_OK) { drain(); return rc; }
        CSF_CUDA_H(cudaEventRecord(c->ev_cmp[s], c->stream));
        CSF_CUDA_H(cudaStreamWaitEvent(c->hs_out, c->ev_cmp[s], 0));
        CSF_CUDA_H(cudaMemcpy2DAsync(hY + v0, (size_t)ld * sizeof(double2), c->h_y[s].p, wbytes, wbytes, rows, cudaMemcpyDeviceToHost, c->hs_out));
        CSF_CUDA_H(cudaEventRecord(c->ev_out[s], c->hs_out));
    }
#undef CSF_CUDA_H
    CSF_CUDA(c, cudaStreamSynchronize(c->hs_out));
    CSF_CUDA(c, cudaStreamSynchronize(c->stream));
    CSF_CUDA(c, cudaStreamSynchronize(c->hs_in));
    return CSF_OK;
    CSF_GUARD_END(c)
}

int csf_set_host_chunk(csf_ctx* c, int ncols) {
    if (!c) return CSF_EINVAL;
    if (ncols < 1) return fail(c, CSF_EINVAL, "host chunk must be >= 1");
    c->host_chunk = ncols;
    return CSF_OK;
}

int csf_profile_enable(csf_ctx* c, int on) { if (!c) return CSF_EINVAL; c->prof = on != 0; return CSF_OK; }

int csf_profile_read(csf_ctx* c, int kind, double* ms_total, int64_t* launches) {
    CSF_GUARD_BEGIN
    if (!c || kind < 0 || kind >= CSF_NKINDS) return CSF_EINVAL;
    CSF_CUDA(c, cudaSetDevice(c->device));
    CSF_CUDA(c, cudaStreamSynchronize(c->stream));
    double tot = 0.0;
    for (auto& pr : c->prof_ev[kind]) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, pr.first, pr.second) == cudaSuccess) tot += ms;
        cudaEventDestroy(pr.first); cudaEventDestroy(pr.second);
    }
    if (ms_total) *ms_total = tot;
    if (launches) *launches = (int64_t)c->prof_ev[kind].size();
    c->prof_ev[kind].clear();
    return CSF_OK;
    CSF_GUARD_END(c)
}

int csf_probe_fp64_peak(int device, double* tflops_fma, double* tflops_mma) {
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return fail(nullptr, CSF_ECUDA, "no such CUDA device");
    if (cudaSetDevice(device) != cudaSuccess) return fail(nullptr, CSF_ECUDA, "cudaSetDevice failed");
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return fail(nullptr, CSF_ECUDA, "cudaGetDeviceProperties failed");
    double* sink = nullptr;
    if (cudaMalloc(&sink, 1 << 20) != cudaSuccess) return fail(nullptr, CSF_ENOMEM, "cudaMalloc failed");
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = prop.multiProcessorCount * 8, iters = 4096;
    double out[2] = {0.0, 0.0};
    for (int which = 0; which < 2; ++which) {
        float best = 1e30f;
        for (int rep = 0; rep < 5; ++rep) {
            cudaEventRecord(e0, 0);
            if (which == 0) probe_dfma_kernel<<<blocks, 256>>>(sink, iters, 1.0000001);
            else probe_dmma_kernel<<<blocks, 256>>>(sink, iters, 1.0000001);
            cudaEventRecord(e1, 0);
            if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(sink); return fail(nullptr, CSF_ECUDA, "probe kernel failed"); }
            float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        // DFMA: 8 chains x 2 flops per iteration per thread; DMMA m8n8k4: 8 mma x 512 flops per iteration per warp
        const double flops = which == 0 ? (double)blocks * 256 * iters * 8 * 2 : (double)blocks * 8 * iters * 8 * 512;
        out[which] = flops / (best * 1e-3) * 1e-12;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    if (tflops_fma) *tflops_fma = out[0];
    if (tflops_mma) *tflops_mma = out[1];
    return CSF_OK;
}

int csf_probe_fp64_mixed(int device, double* tflops_total) {
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return fail(nullptr, CSF_ECUDA, "no such CUDA device");
    if (cudaSetDevice(device) != cudaSuccess) return fail(nullptr, CSF_ECUDA, "cudaSetDevice failed");
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return fail(nullptr, CSF_ECUDA, "cudaGetDeviceProperties failed");
    double* sink = nullptr;
    if (cudaMalloc(&sink, 1 << 20) != cudaSuccess) return fail(nullptr, CSF_ENOMEM, "cudaMalloc failed");
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = prop.multiProcessorCount * 4, iters = 4096;
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, 0);
        probe_mixed_kernel<<<blocks, 256>>>(sink, iters, 1.0000001);
        cudaEventRecord(e1, 0);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(sink); return fail(nullptr, CSF_ECUDA, "probe kernel failed"); }
        float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    // per CTA: 4 warps x 32 threads x 8 chains x 2 flops (DFMA) + 4 warps x 8 mma x 512 flops (DMMA) per iteration
    const double flops = (double)blocks * iters * (4.0 * 32 * 8 * 2 + 4.0 * 8 * 512);
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    if (tflops_total) *tflops_total = flops / (best * 1e-3) * 1e-12;
    return CSF_OK;
}

int csf_column_lanes(const csf_ctx* c, int nvec, int mode, int* lanes) {
    if (!c || !lanes || nvec < 1 || (mode != CSF_FP64 && mode != CSF_FP32_INTERMEDIATE)) return CSF_EINVAL;
    const bool f32 = mode == CSF_FP32_INTERMEDIATE;
    *lanes = column_info(c->p, column_kind(c)).lanes;
    return CSF_OK;
}

int csf_filter_fused_gather(const csf_ctx* c, int nvec, int mode, int* fused) {
    if (!c || !fused || nvec < 1 || (mode != CSF_FP64 && mode != CSF_FP32_INTERMEDIATE)) return CSF_EINVAL;
    *fused = (mode == CSF_FP64 && !c->kpt_on && !c->proj_complex && fused_gather_ok(c, nvec)) ? 1 : 0;
    return CSF_OK;
}

int csf_launch_count(const csf_ctx* c, int64_t* launches) { if (!c || !launches) return CSF_EINVAL; *launches = c->launches; return CSF_OK; }

int csf_set_tuning(csf_ctx* c, int seg_len, int chunk_group) {
    if (!c) return CSF_EINVAL;
    if (seg_len < 0 || chunk_group < 1) return fail(c, CSF_EINVAL, "need seg_len >= 0 and chunk_group >= 1");
    c->seg_len = seg_len; c->chunk_group = chunk_group;
    return CSF_OK;
}

int csf_set_variant(csf_ctx* c, int variant) {
    if (!c) return CSF_EINVAL;
    if (variant < 0 || variant > 1) return fail(c, CSF_EINVAL, "unknown variant");
    c->variant = variant;
    return CSF_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------------------------
// Subspace steps around the filter: Rayleigh-Ritz, density / magnetisation, Lanczos
// ------------------------------------------------------------------------------------------------------------------
namespace {

size_t rr_gram_bytes(int nvec) { return ((size_t)4 * nvec * nvec * sizeof(double) + 255) / 256 * 256; }      // real [2N][2N]

// G = A^T B as real matrices, then the complex nvec x nvec result into dOut (row-major)
int enqueue_gram(csf_ctx* c, const double* A, long long lda, const double* B, long long ldb, int nvec, double* dG, double2* dOut, int sym) {
    static bool configured[64] = {};
    int dev = 0; CSF_CUDA(c, cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        CSF_CUDA(c, cudaFuncSetAttribute(gram_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kGramSmem));
        CSF_CUDA(c, cudaFuncSetAttribute(rotate_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRotSmem));
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    const long long rows = 2 * c->M; const int nc = 2 * nvec, nt = (nc + kGT - 1) / kGT;
    CSF_CUDA(c, cudaMemsetAsync(dG, 0, (size_t)nc * nc * sizeof(double), c->stream));
    // row ranges: enough CTAs for ~4 waves of 2 CTAs per SM over the (upper-triangle) tiles
    // (128 x 128 output tiles — 32 x 64 per warp, twice the flops per byte read from L2, but 168 registers and 135 KB of shared
    // memory, i.e. one CTA of 8 warps per SM — measured 253 against 212 ms for the two projections at config 3: dropped)
    const int tiles = sym ? nt * (nt + 1) / 2 : nt * nt;
    long long nsplit = std::max<long long>(1, std::min<long long>((8LL * c->sm_count + tiles - 1) / tiles, (rows + 4 * kGK - 1) / (4 * kGK)));
    nsplit = std::min<long long>(nsplit, 65535);
    const long long rpc = ((rows + nsplit - 1) / nsplit + kGK - 1) / kGK * kGK;
    dim3 grid(nt * nt, (unsigned)((rows + rpc - 1) / rpc));
    { ProfScope ps(c, CSF_KIND_AUX); gram_kernel<<<grid, 256, kGramSmem, c->stream>>>(A, lda, B, ldb, nc, rows, rpc, dG, nc, sym); }
    CSF_CUDA(c, cudaGetLastError());
    gram_finish_kernel<<<(nvec * nvec + 255) / 256, 256, 0, c->stream>>>(dG, nc, nvec, dOut, nvec, sym);
    CSF_CUDA(c, cudaGetLastError());
    c->launches += 2;
    return CSF_OK;
}

// cuSOLVER's dense Hermitian-definite eigensolver, resolved at first use (no link-time dependency)
struct CuSolver {
    void* lib = nullptr;
    cusolverStatus_t (*create)(cusolverDnHandle_t*) = nullptr;
    cusolverStatus_t (*destroy)(cusolverDnHandle_t) = nullptr;
    cusolverStatus_t (*set_stream)(cusolverDnHandle_t, cudaStream_t) = nullptr;
    cusolverStatus_t (*bufsize)(cusolverDnHandle_t, cusolverEigType_t, cusolverEigMode_t, cublasFillMode_t, int, const cuDoubleComplex*, int, const cuDoubleComplex*, int, const double*, int*) = nullptr;
    cusolverStatus_t (*hegvd)(cusolverDnHandle_t, cusolverEigType_t, cusolverEigMode_t, cublasFillMode_t, int, cuDoubleComplex*, int, cuDoubleComplex*, int, double*, cuDoubleComplex*, int, int*) = nullptr;
    bool load() {
        if (hegvd) return true;
        for (const char* name : {"libcusolver.so.11", "libcusolver.so", "/usr/local/cuda/lib64/libcusolver.so.11"}) { lib = dlopen(name, RTLD_NOW | RTLD_GLOBAL); if (lib) break; }
        if (!lib) return false;
        create = reinterpret_cast<decltype(create)>(dlsym(lib, "cusolverDnCreate"));
        destroy = reinterpret_cast<decltype(destroy)>(dlsym(lib, "cusolverDnDestroy"));
        set_stream = reinterpret_cast<decltype(set_stream)>(dlsym(lib, "cusolverDnSetStream"));
        bufsize = reinterpret_cast<decltype(bufsize)>(dlsym(lib, "cusolverDnZhegvd_bufferSize"));
        hegvd = reinterpret_cast<decltype(hegvd)>(dlsym(lib, "cusolverDnZhegvd"));
        return create && destroy && set_stream && bufsize && hegvd;
    }
} g_cusolver;

// dst[i][j] = conj(src[j][i]) (n x n)
__global__ void __launch_bounds__(256) conj_transpose_kernel(const double2* __restrict__ src, double2* __restrict__ dst, int n) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n * n) return;
    const int i = idx / n, j = idx % n; const double2 z = src[(long long)j * n + i];
    dst[idx] = make_double2(z.x, -z.y);
}
__global__ void __launch_bounds__(256) recip_kernel(const double* __restrict__ a, double* __restrict__ o, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) o[i] = 1.0 / a[i];
}

}  // namespace

extern "C" {

static int enqueue_dense_step(csf_ctx* c, const double2* src, long long ld, double* dst, long long ld_dst, int nvec, double sc, int rot, double shift, char* coef);

// Scratch of one H apply with whichever operator the context holds, and the apply itself (dst += Hhat src): the sum-factorised
// Gamma-point operator, or, while a k-point / complex projectors are set, the dense-path operator Hhat^k (csf_dense.cuh)
static size_t apply_scratch_bytes(const csf_ctx* c, int nvec) { return std::max(coef_bytes(c, nvec) + ctp_bytes(c, nvec), 3 * coef_bytes(c, nvec)); }
static bool dense_only(const csf_ctx* c) { return c->kpt_on || c->proj_complex; }
static int enqueue_apply(csf_ctx* c, const void* src, long long ld, double* dst, long long ld_dst, int nvec, char* scratch) {
    if (dense_only(c)) {
        if (c->dense_nq == 0) return fail(c, CSF_ESTATE, "csf_set_potential_quadrature has not been called (it must follow csf_set_kpoint)");
        return enqueue_dense_step(c, static_cast<const double2*>(src), ld, dst, ld_dst, nvec, 1.0, 0, 0.0, scratch);
    }
    return enqueue_step(c, src, ld, dst, ld_dst, nvec, 1.0, 0, 0.0, reinterpret_cast<double*>(scratch), reinterpret_cast<double*>(scratch + coef_bytes(c, nvec)));
}

int csf_rr_workspace_bytes(const csf_ctx* c, int nvec, size_t* bytes) {
    if (!c || !bytes || nvec < 0) return CSF_EINVAL;
    *bytes = block_bytes(c, nvec) + apply_scratch_bytes(c, nvec) + rr_gram_bytes(nvec) + 256;
    return CSF_OK;
}

int csf_rr_project(csf_ctx* c, const csf_c128* dX, int64_t ld, int nvec, csf_c128* dHs, csf_c128* dSs, void* d_work, size_t work_bytes) {
    if (!c) return CSF_EINVAL;
    CSF_GUARD_BEGIN
    if (!dHs || !dSs) return fail(c, CSF_EINVAL, "NULL output pointer");
    size_t need = 0; csf_rr_workspace_bytes(c, std::max(nvec, 0), &need);
    int rc = check_block_args(c, dX, dHs, ld, nvec, d_work, work_bytes, need);
    if (rc != CSF_OK || nvec == 0) return rc;
    CSF_CUDA(c, cudaSetDevice(c->device));
    char* w = static_cast<char*>(d_work);
    double* HX = reinterpret_cast<double*>(w);                                        // [2M][nvec] complex128
    char* scratch = w + block_bytes(c, nvec);
    double* dG = reinterpret_cast<double*>(w + block_bytes(c, nvec) + apply_scratch_bytes(c, nvec));
    rc = enqueue_zero(c, HX, nvec, nvec); if (rc != CSF_OK) return rc;
    rc = enqueue_apply(c, dX, ld, HX, nvec, nvec, scratch); if (rc != CSF_OK) return rc;
    const double* Xr = reinterpret_cast<const double*>(dX);
    rc = enqueue_gram(c, Xr, 2 * ld, HX, 2LL * nvec, nvec, dG, reinterpret_cast<double2*>(dHs), 1); if (rc != CSF_OK) return rc;      // Hs = X^dagger (Hhat X)
    return enqueue_gram(c, Xr, 2 * ld, Xr, 2 * ld, nvec, dG, reinterpret_cast<double2*>(dSs), 1);                                   // Ss = X^dagger X
    CSF_GUARD_END(c)
}

int csf_rr_solve(csf_ctx* c, const csf_c128* dHs, const csf_c128* dSs, int n, csf_c128* dQ, double* lambda_host) {
    if (!c) return CSF_EINVAL;
    CSF_GUARD_BEGIN
    if (!dHs || !dSs || !dQ || !lambda_host || n < 1) return fail(c, CSF_EINVAL, "bad argument");
    CSF_CUDA(c, cudaSetDevice(c->device));
    if (!g_cusolver.load()) return fail(c, CSF_EUNSUPPORTED, "libcusolver not found");
    cusolverDnHandle_t h = nullptr;
    if (g_cusolver.create(&h) != CUSOLVER_STATUS_SUCCESS) return fail(c, CSF_ECUDA, "cusolverDnCreate failed");
    g_cusolver.set_stream(h, c->stream);
    // The row-major Hermitian matrices are the conjugates of the column-major ones cuSOLVER sees: conj(Hs) y = lambda conj(Ss) y,
    // so the wanted eigenvectors are q = conj(y), and Q[i][j] = q_j[i] = conj(V_colmajor(i, j)): a conjugate transpose of the buffer.
    DevBuf a, b, wv, work, info;
    const size_t nn = (size_t)n * n * sizeof(double2);
    int rc = CSF_OK;
    cudaError_t e = a.alloc(nn); if (e == cudaSuccess) e = b.alloc(nn); if (e == cudaSuccess) e = wv.alloc((size_t)n * sizeof(double)); if (e == cudaSuccess) e = info.alloc(sizeof(int));
    if (e != cudaSuccess) { g_cusolver.destroy(h); return cuda_fail(c, e, "cudaMalloc"); }
    cudaMemcpyAsync(a.p, dHs, nn, cudaMemcpyDeviceToDevice, c->stream); cudaMemcpyAsync(b.p, dSs, nn, cudaMemcpyDeviceToDevice, c->stream);
    int lwork = 0;
    if (g_cusolver.bufsize(h, CUSOLVER_EIG_TYPE_1, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, n, a.as<cuDoubleComplex>(), n, b.as<cuDoubleComplex>(), n, wv.as<double>(), &lwork) != CUSOLVER_STATUS_SUCCESS)
        rc = fail(c, CSF_ECUDA, "cusolverDnZhegvd_bufferSize failed");
    if (rc == CSF_OK && work.alloc((size_t)std::max(lwork, 1) * sizeof(double2)) != cudaSuccess) rc = fail(c, CSF_ENOMEM, "cudaMalloc failed");
    if (rc == CSF_OK && g_cusolver.hegvd(h, CUSOLVER_EIG_TYPE_1, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, n, a.as<cuDoubleComplex>(), n, b.as<cuDoubleComplex>(), n,
                                         wv.as<double>(), work.as<cuDoubleComplex>(), lwork, info.as<int>()) != CUSOLVER_STATUS_SUCCESS)
        rc = fail(c, CSF_ECUDA, "cusolverDnZhegvd failed");
    int hinfo = 0;
    if (rc == CSF_OK) {
        conj_transpose_kernel<<<(n * n + 255) / 256, 256, 0, c->stream>>>(a.as<double2>(), reinterpret_cast<double2*>(dQ), n);
        cudaMemcpyAsync(lambda_host, wv.p, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
        cudaMemcpyAsync(&hinfo, info.p, sizeof(int), cudaMemcpyDeviceToHost, c->stream);
        e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) rc = cuda_fail(c, e, "csf_rr_solve");
        else if (hinfo != 0) rc = fail(c, CSF_EINVAL, hinfo > n ? "X^dagger X is not positive definite (linearly dependent block)" : "eigensolver did not converge");
    } else cudaStreamSynchronize(c->stream);
    g_cusolver.destroy(h);
    return rc;
    CSF_GUARD_END(c)
}

int csf_rr_rotate(csf_ctx* c, const csf_c128* dX, int64_t ld, int nvec, const csf_c128* dQ, csf_c128* dU, int64_t ldu, void* d_work, size_t work_bytes) {
    if (!c) return CSF_EINVAL;
    CSF_GUARD_BEGIN
    if (!dQ) return fail(c, CSF_EINVAL, "Q is NULL");
    if (ldu < nvec) return fail(c, CSF_EINVAL, "need ldu >= nvec");
    int rc = check_block_args(c, dX, dU, ld, nvec, d_work, work_bytes, rr_gram_bytes(std::max(nvec, 0)));
    if (rc != CSF_OK || nvec == 0) return rc;
    CSF_CUDA(c, cudaSetDevice(c->device));
    double* Qt = static_cast<double*>(d_work);
    const int k2 = 2 * nvec; const long long rows = 2 * c->M;
    qtilde_kernel<<<(nvec * nvec + 255) / 256, 256, 0, c->stream>>>(reinterpret_cast<const double2*>(dQ), nvec, nvec, Qt, k2);
    CSF_CUDA(c, cudaGetLastError());
    static bool configured[64] = {};
    int dev = 0; CSF_CUDA(c, cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        CSF_CUDA(c, cudaFuncSetAttribute(rotate_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRotSmem));
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    const long long rt = (rows + kGT - 1) / kGT, nct = (k2 + kGT - 1) / kGT;
    if (rt * nct > 0x7fffffffLL) return fail(c, CSF_EUNSUPPORTED, "grid too large");
    { ProfScope ps(c, CSF_KIND_AUX); rotate_kernel<<<(unsigned)(rt * nct), 256, kRotSmem, c->stream>>>(reinterpret_cast<const double*>(dX), 2 * ld, Qt, k2, k2, reinterpret_cast<double*>(dU), 2 * ldu, rows); }
    CSF_CUDA(c, cudaGetLastError());
    c->launches += 2;
    return CSF_OK;
    CSF_GUARD_END(c)
}

int csf_density(csf_ctx* c, const csf_c128* dX, int64_t ld, int nvec, const double* occ_host, double* d_rho_m, int accumulate) {
    if (!c) return CSF_EINVAL;
    CSF_GUARD_BEGIN
    if (!dX || !occ_host || !d_rho_m) return fail(c, CSF_EINVAL, "NULL argument");
    if (nvec < 0 || ld < nvec) return fail(c, CSF_EINVAL, "need 0 <= nvec <= ld");
    CSF_CUDA(c, cudaSetDevice(c->device));
    if (!c->d_inv_mass.p) {
        std::vector<double> mass((size_t)c->M);
        csf_mass_diag(c, mass.data());
        DevBuf tmp; CSF_CUDA(c, tmp.upload(mass));
        CSF_CUDA(c, c->d_inv_mass.alloc((size_t)c->M * sizeof(double)));
        recip_kernel<<<(unsigned)((c->M + 255) / 256), 256, 0, c->stream>>>(tmp.as<double>(), c->d_inv_mass.as<double>(), c->M);
        CSF_CUDA(c, cudaStreamSynchronize(c->stream));
    }
    if (nvec == 0) { if (!accumulate) CSF_CUDA(c, cudaMemsetAsync(d_rho_m, 0, (size_t)c->M * 4 * sizeof(double), c->stream)); return CSF_OK; }
    if (c->d_occ.bytes < (size_t)nvec * sizeof(double)) CSF_CUDA(c, c->d_occ.alloc((size_t)nvec * sizeof(double)));
    CSF_CUDA(c, cudaMemcpyAsync(c->d_occ.p, occ_host, (size_t)nvec * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    CSF_CUDA(c, cudaStreamSynchronize(c->stream));                  // occ_host may be pageable and go out of scope
    { ProfScope ps(c, CSF_KIND_AUX); density_kernel<<<(unsigned)((c->M + 7) / 8), 256, 0, c->stream>>>(reinterpret_cast<const double2*>(dX), ld, nvec, c->d_occ.as<double>(), c->d_inv_mass.as<double>(), c->M, d_rho_m, accumulate); }
    CSF_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return CSF_OK;
    CSF_GUARD_END(c)
}

int csf_lanczos_workspace_bytes(const csf_ctx* c, size_t* bytes) {
    if (!c || !bytes) return CSF_EINVAL;
    *bytes = 3 * block_bytes(c, 1) + apply_scratch_bytes(c, 1) + 512;
    return CSF_OK;
}

int csf_lanczos(csf_ctx* c, const csf_c128* d_v0, int k, double* alpha_host, double* beta_host, int* steps_done, void* d_work, size_t work_bytes) {
    if (!c) return CSF_EINVAL;
    CSF_GUARD_BEGIN
    if (!d_v0 || !alpha_host || !beta_host || k < 1) return fail(c, CSF_EINVAL, "bad argument");
    if (!c->have_pot && !dense_only(c)) return fail(c, CSF_ESTATE, "csf_set_potential has not been called");
    size_t need = 0; csf_lanczos_workspace_bytes(c, &need);
    if (!d_work || work_bytes < need) return fail(c, CSF_EINVAL, "workspace too small");
    CSF_CUDA(c, cudaSetDevice(c->device));
    const long long n = 2 * c->M; const size_t vb = block_bytes(c, 1);
    char* w8 = static_cast<char*>(d_work);
    double2* v = reinterpret_cast<double2*>(w8); double2* vprev = reinterpret_cast<double2*>(w8 + vb); double2* w = reinterpret_cast<double2*>(w8 + 2 * vb);
    char* apply_scratch = w8 + 3 * vb;
    double* scratch = reinterpret_cast<double*>(w8 + 3 * vb + apply_scratch_bytes(c, 1));
    const int grid = c->sm_count * 8;
    double hs[2] = {0.0, 0.0};
    // v = v0 / |v0|, vprev = 0
    CSF_CUDA(c, cudaMemsetAsync(scratch, 0, 2 * sizeof(double), c->stream));
    CSF_CUDA(c, cudaMemsetAsync(v, 0, vb, c->stream));
    CSF_CUDA(c, cudaMemcpyAsync(w, d_v0, vb, cudaMemcpyDeviceToDevice, c->stream));
    lanczos_b_kernel<<<grid, 256, 0, c->stream>>>(w, v, 0.0, n, scratch);
    CSF_CUDA(c, cudaMemcpyAsync(hs, scratch, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CSF_CUDA(c, cudaStreamSynchronize(c->stream));
    if (!(hs[1] > 0.0)) return fail(c, CSF_EINVAL, "start vector is zero");
    lanczos_c_kernel<<<grid, 256, 0, c->stream>>>(vprev, v, w, 1.0 / std::sqrt(hs[1]), n);        // vprev = 0, v = v0 / |v0|
    double beta = 0.0; int done = 0;
    for (int j = 0; j < k; ++j) {
        int rc = enqueue_zero(c, reinterpret_cast<double*>(w), 1, 1); if (rc != CSF_OK) return rc;
        rc = enqueue_apply(c, v, 1, reinterpret_cast<double*>(w), 1, 1, apply_scratch); if (rc != CSF_OK) return rc;
        CSF_CUDA(c, cudaMemsetAsync(scratch, 0, 2 * sizeof(double), c->stream));
        lanczos_a_kernel<<<grid, 256, 0, c->stream>>>(w, vprev, v, beta, n, scratch);
        CSF_CUDA(c, cudaMemcpyAsync(hs, scratch, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        CSF_CUDA(c, cudaStreamSynchronize(c->stream));
        const double alpha = hs[0];
        lanczos_b_kernel<<<grid, 256, 0, c->stream>>>(w, v, alpha, n, scratch);
        CSF_CUDA(c, cudaMemcpyAsync(hs, scratch, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        CSF_CUDA(c, cudaStreamSynchronize(c->stream));
        beta = std::sqrt(hs[1]);
        alpha_host[j] = alpha; beta_host[j] = beta; done = j + 1;
        c->launches += 3;
        if (!(beta > 1e-300)) break;
        lanczos_c_kernel<<<grid, 256, 0, c->stream>>>(vprev, v, w, 1.0 / beta, n);
    }
    CSF_CUDA(c, cudaGetLastError());
    if (steps_done) *steps_done = done;
    return CSF_OK;
    CSF_GUARD_END(c)
}

int csf_tridiag_extremes(const double* alpha, const double* beta, int k, double* theta_min, double* theta_max) {
    if (!alpha || !beta || k < 1 || !theta_min || !theta_max) return CSF_EINVAL;
    // Sturm-sequence bisection on the symmetric tridiagonal matrix (alpha, beta[0..k-2]); Gershgorin interval first
    double lo = alpha[0], hi = alpha[0];
    for (int i = 0; i < k; ++i) {
        const double r = (i > 0 ? std::fabs(beta[i - 1]) : 0.0) + (i + 1 < k ? std::fabs(beta[i]) : 0.0);
        lo = std::min(lo, alpha[i] - r); hi = std::max(hi, alpha[i] + r);
    }
    auto count_below = [&](double x) {                 // number of eigenvalues < x
        int cnt = 0; double d = 1.0;
        for (int i = 0; i < k; ++i) {
            const double b2 = i > 0 ? beta[i - 1] * beta[i - 1] : 0.0;
            d = alpha[i] - x - (i > 0 ? b2 / d : 0.0);
            if (d == 0.0) d = -1e-300;
            if (d < 0.0) ++cnt;
        }
        return cnt;
    };
    auto kth = [&](int idx) {                          // eigenvalue number idx (0-based, ascending)
        double a = lo, b = hi;
        for (int it = 0; it < 200 && b - a > 4e-16 * std::max(std::fabs(a), std::fabs(b)); ++it) {
            const double m = 0.5 * (a + b);
            if (count_below(m) > idx) b = m; else a = m;
        }
        return 0.5 * (a + b);
    };
    *theta_min = kth(0); *theta_max = kth(k - 1);
    return CSF_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// potential at the Gauss-Legendre points of an n_q^3 rule (eq.79-83) and the dense
// cell-matrix form of H X (eq.84); kernels in csf_dense.cuh

int csf_quadrature_points(const csf_ctx* c, int nq, double* xyz) {
    CSF_GUARD_BEGIN
    if (!c || !xyz) return CSF_EINVAL;
    double x[kMaxQ], w[kMaxQ];
    if (!build_gauss_legendre(nq, x, w)) return fail(const_cast<csf_ctx*>(c), CSF_EINVAL, "need 1 <= nq <= 16");
    const long long nq3 = (long long)nq * nq * nq;
    for (long long e = 0; e < c->E; ++e) {
        const int cc[3] = {(int)(e % c->ncell[0]), (int)((e / c->ncell[0]) % c->ncell[1]), (int)(e / ((long long)c->ncell[0] * c->ncell[1]))};
        for (int qz = 0; qz < nq; ++qz) for (int qy = 0; qy < nq; ++qy) for (int qx = 0; qx < nq; ++qx) {
            double* o = xyz + (e * nq3 + qx + nq * (qy + (long long)nq * qz)) * 3;
            o[0] = (cc[0] + 0.5 * (x[qx] + 1.0)) * c->h[0]; o[1] = (cc[1] + 0.5 * (x[qy] + 1.0)) * c->h[1]; o[2] = (cc[2] + 0.5 * (x[qz] + 1.0)) * c->h[2];
        }
    }
    return CSF_OK;
    CSF_GUARD_END(c)
}

int csf_set_potential_quadrature(csf_ctx* c, int nq, const double* vq) {
    CSF_GUARD_BEGIN
    if (!c) return CSF_EINVAL;
    if (!vq) return fail(c, CSF_EINVAL, "vq is NULL");
    double gx[kMaxQ], gw[kMaxQ];
    if (!build_gauss_legendre(nq, gx, gw)) return fail(c, CSF_EINVAL, "need 1 <= nq <= 16");
    CSF_CUDA(c, cudaSetDevice(c->device));
    const int n = c->n, n3 = n * n * n, n3p = (n3 + 7) / 8 * 8, nq3 = nq * nq * nq;
    const size_t mat_bytes = (size_t)c->E * 4 * n3p * n3p * sizeof(double);
    size_t free_b = 0, total_b = 0;
    CSF_CUDA(c, cudaMemGetInfo(&free_b, &total_b));
    const size_t have = c->d_cellmat.bytes, reserve = (size_t)256 << 20;          // (the old matrices are released before the new ones are allocated)
    if (mat_bytes > have && mat_bytes - have + reserve > free_b)
        return fail(c, CSF_ENOMEM, "dense cell matrices need " + std::to_string(mat_bytes) + " bytes of device memory (4 n_p^6 doubles per cell); " + std::to_string(free_b) + " free");
    // 1-D tables: L[i][q] = l_i(x_q), s_i = m1d_i^(-1/2) per direction
    std::vector<double> L((size_t)n * nq);
    lagrange_at_points(c->gll, nq, gx, L.data());
    std::vector<double> Ns((size_t)nq3 * n3p, 0.0), wJ((size_t)nq3), kin((size_t)n3p * n3p, 0.0);
    const double J = c->h[0] * c->h[1] * c->h[2] / 8.0;
    for (int qz = 0; qz < nq; ++qz) for (int qy = 0; qy < nq; ++qy) for (int qx = 0; qx < nq; ++qx) {
        const size_t q = qx + (size_t)nq * (qy + (size_t)nq * qz);
        wJ[q] = gw[qx] * gw[qy] * gw[qz] * J;
        for (int k = 0; k < n; ++k) for (int j = 0; j < n; ++j) for (int i = 0; i < n; ++i) {
            const double s = 1.0 / std::sqrt(c->dir[0].m1d[i] * c->dir[1].m1d[j] * c->dir[2].m1d[k]);
            Ns[q * n3p + i + n * (j + n * k)] = s * L[(size_t)i * nq + qx] * L[(size_t)j * nq + qy] * L[(size_t)k * nq + qz];
        }
    }
    // S 1/2 K^(e) S = Bz (x) By (x) Ax + Bz (x) Ay (x) Bx + Az (x) By (x) Bx with B = diag(beta) - u u^T (csf_tables.h; eq.40 first term)
    auto Bm = [&](int d, int i, int j) { return (i == j ? c->dir[d].beta[i] : 0.0) - c->dir[d].u[i] * c->dir[d].u[j]; };
    for (int k = 0; k < n; ++k) for (int j = 0; j < n; ++j) for (int i = 0; i < n; ++i)
        for (int k2 = 0; k2 < n; ++k2) for (int j2 = 0; j2 < n; ++j2) for (int i2 = 0; i2 < n; ++i2) {
            const double bx = Bm(0, i, i2), by = Bm(1, j, j2), bz = Bm(2, k, k2);
            kin[(size_t)(i + n * (j + n * k)) * n3p + i2 + n * (j2 + n * k2)] =
                bz * by * c->dir[0].A[i][i2] + bz * c->dir[1].A[j][j2] * bx + c->dir[2].A[k][k2] * by * bx;
        }
    DevBuf dNs, dwJ, dkin, dvq; double cp_vshift = 0.0;
    CSF_CUDA(c, cudaStreamSynchronize(c->stream));
    CSF_CUDA(c, dNs.upload(Ns)); CSF_CUDA(c, dwJ.upload(wJ)); CSF_CUDA(c, dkin.upload(kin));
    CSF_CUDA(c, dvq.alloc((size_t)c->E * nq3 * 4 * sizeof(double)));
    CSF_CUDA(c, cudaMemcpy(dvq.p, vq, (size_t)c->E * nq3 * 4 * sizeof(double), cudaMemcpyHostToDevice));
    cp_vshift = 0.5 * (c->kpt[0] * c->kpt[0] + c->kpt[1] * c->kpt[1] + c->kpt[2] * c->kpt[2]);      // |k|^2/2 stands beside V_eff in eq.40 (reading A19)
    if (c->d_cellmat.bytes != mat_bytes) { if (c->d_cellmat.alloc(mat_bytes) != cudaSuccess) { cudaGetLastError(); c->dense_nq = 0; return fail(c, CSF_ENOMEM, "cudaMalloc of the dense cell matrices failed"); } }
    CellMatParams cp{};
    cp.Ns = dNs.as<double>(); cp.wJ = dwJ.as<double>(); cp.kin = dkin.as<double>(); cp.vq = dvq.as<double>(); cp.out = c->d_cellmat.as<double>();
    cp.nq3 = nq3; cp.n3 = n3; cp.n3p = n3p; cp.vshift = cp_vshift;
    const long long nblk = (long long)c->E * (n3p / 8);
    if (nblk > 0x7fffffffLL) return fail(c, CSF_EUNSUPPORTED, "grid too large");
    cellmat_build_kernel<<<(unsigned)nblk, 256, 0, c->stream>>>(cp);
    CSF_CUDA(c, cudaGetLastError());
    CSF_CUDA(c, cudaStreamSynchronize(c->stream));        // the staging buffers above are freed on return
    c->dense_nq = nq; c->dense_n3p = n3p; c->launches += 1;
    return CSF_OK;
    CSF_GUARD_END(c)
}

int csf_set_kpoint(csf_ctx* c, const double* k) {
    CSF_GUARD_BEGIN
    if (!c || !k) return CSF_EINVAL;
    CSF_CUDA(c, cudaSetDevice(c->device));
    CSF_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int d = 0; d < 3; ++d) c->kpt[d] = k[d];
    c->kpt_on = k[0] != 0.0 || k[1] != 0.0 || k[2] != 0.0;
    c->dense_nq = 0;                          // the cell matrices carry |k|^2/2: csf_set_potential_quadrature must follow
    if (!c->kpt_on) { c->d_gk.release(); return CSF_OK; }
    // S sum_d k_d G_d^(e) S with G_x = Mz (x) My (x) Gx: the scaled 1-D mass B = diag(beta) - u u^T (csf_tables.h) and the scaled
    // 1-D gradient C_ij = s_i w_i D_ij s_j (int l_i l_j' = w_i D_ij exactly; the (2/h)(h/2) of the derivative and the measure cancel)
    const int n = c->n, n3 = n * n * n, n3p = (n3 + 7) / 8 * 8, ksn = n3p / 4;
    auto Bm = [&](int d, int i, int j) { return (i == j ? c->dir[d].beta[i] : 0.0) - c->dir[d].u[i] * c->dir[d].u[j]; };
    auto Cm = [&](int d, int i, int j) { return c->gll.w[i] * c->gll.D[i][j] / std::sqrt(c->dir[d].m1d[i] * c->dir[d].m1d[j]); };
    std::vector<double> gk((size_t)n3p * n3p, 0.0);
    for (int kz = 0; kz < n; ++kz) for (int j = 0; j < n; ++j) for (int i = 0; i < n; ++i)
        for (int k2 = 0; k2 < n; ++k2) for (int j2 = 0; j2 < n; ++j2) for (int i2 = 0; i2 < n; ++i2) {
            const double bx = Bm(0, i, i2), by = Bm(1, j, j2), bz = Bm(2, kz, k2);
            const double v = k[0] * bz * by * Cm(0, i, i2) + k[1] * bz * Cm(1, j, j2) * bx + k[2] * Cm(2, kz, k2) * by * bx;
            const int a = i + n * (j + n * kz), b = i2 + n * (j2 + n * k2);
            gk[((size_t)(a / 8) * ksn + b / 4) * 32 + (a % 8) * 4 + b % 4] = v;
        }
    CSF_CUDA(c, c->d_gk.upload(gk));
    return CSF_OK;
    CSF_GUARD_END(c)
}

int csf_dense_workspace_bytes(const csf_ctx* c, int nvec, size_t* bytes) {
    if (!c || !bytes || nvec < 0) return CSF_EINVAL;
    // one block buffer for the recurrence of csf_filter_dense + C (and the second gather of complex projectors) + Delta C
    *bytes = block_bytes(c, nvec) + (c->natoms > 0 ? 3 * coef_bytes(c, nvec) : 0) + 256;
    return CSF_OK;
}

// dst += sc i^rot (Hhat^k - shift) src through the dense cell matrices; coef: 3 coef_bytes of workspace (unused without projectors)
static int enqueue_dense_step(csf_ctx* c, const double2* src, long long ld, double* dst, long long ld_dst, int nvec, double sc, int rot, double shift, char* coef) {
    const double frs[4] = {1.0, 0.0, -1.0, 0.0}, fis[4] = {0.0, 1.0, 0.0, -1.0};
    const double fr = sc * frs[rot & 3], fi = sc * fis[rot & 3];
    DenseParams q{};
    q.mat = c->d_cellmat.as<double>(); q.X = src; q.ld = ld; q.Y = dst; q.ldy = ld_dst;
    q.nvec = nvec; q.p = c->p; q.n3 = c->n * c->n * c->n; q.n3p = c->dense_n3p;
    q.ncx = c->ncell[0]; q.ncy = c->ncell[1]; q.ncz = c->ncell[2]; q.nfx = c->nfree[0]; q.nfy = c->nfree[1]; q.nfz = c->nfree[2];
    q.bcx = c->bc[0] == CSF_BC_DIRICHLET; q.bcy = c->bc[1] == CSF_BC_DIRICHLET; q.bcz = c->bc[2] == CSF_BC_DIRICHLET;
    q.fr = fr; q.fi = fi; q.gk = c->d_gk.as<double>();
    // 16 vectors per CTA where the X tile of the cell still leaves room for two CTAs per SM (up to order 5), 8 otherwise
    const bool v16 = nvec > 8 && 2 * (dense_smem<16>(q.n3p) + 1024) <= 227 * 1024;
    const int vc = v16 ? 16 : 8;
    const size_t smem = v16 ? dense_smem<16>(q.n3p) : dense_smem<8>(q.n3p);
    if (smem > c->smem_optin) return fail(c, CSF_EUNSUPPORTED, "cell tile does not fit shared memory");
    const long long nblk = (long long)c->E * ((nvec + vc - 1) / vc);
    if (nblk > 0x7fffffffLL) return fail(c, CSF_EUNSUPPORTED, "grid too large");
    {
        static bool configured[64] = {};
        if (c->device >= 64 || !configured[c->device]) {
            CSF_CUDA(c, cudaFuncSetAttribute(dense_cell_kernel<8, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_optin));
            CSF_CUDA(c, cudaFuncSetAttribute(dense_cell_kernel<16, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_optin));
            CSF_CUDA(c, cudaFuncSetAttribute(dense_cell_kernel<8, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_optin));
            CSF_CUDA(c, cudaFuncSetAttribute(dense_cell_kernel<16, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_optin));
            if (c->device < 64) configured[c->device] = true;
        }
        ProfScope ps(c, CSF_KIND_CELL);
        if (c->kpt_on) { if (v16) dense_cell_kernel<16, true><<<(unsigned)nblk, 256, smem, c->stream>>>(q); else dense_cell_kernel<8, true><<<(unsigned)nblk, 256, smem, c->stream>>>(q); }
        else { if (v16) dense_cell_kernel<16, false><<<(unsigned)nblk, 256, smem, c->stream>>>(q); else dense_cell_kernel<8, false><<<(unsigned)nblk, 256, smem, c->stream>>>(q); }
    }
    CSF_CUDA(c, cudaGetLastError());
    c->launches += 1;
    if (shift != 0.0) {
        ProfScope ps(c, CSF_KIND_AUX);
        caxpy_kernel<<<c->sm_count * 8, 256, 0, c->stream>>>(src, ld, reinterpret_cast<double2*>(dst), ld_dst, 2 * c->M, nvec, -fr * shift, -fi * shift);
        CSF_CUDA(c, cudaGetLastError());
        c->launches += 1;
    }
    if (c->natoms == 0) return CSF_OK;
    // step 4: dst += f P~ Delta P~^+ src, P~ = Re + i Im
    const size_t cb = coef_bytes(c, nvec);
    double* dC = reinterpret_cast<double*>(coef);
    double* dC2 = reinterpret_cast<double*>(coef + cb);
    double2* dD = reinterpret_cast<double2*>(coef + 2 * cb);
    const long long ldc = nvec;
    CSF_CUDA(c, cudaMemsetAsync(dC, 0, (c->proj_complex ? 2 : 1) * cb, c->stream));
    GatherParams gp{};
    gp.src = src; gp.ld = ld; gp.nvec = nvec;
    gp.gb_atom = c->d_gb_atom.as<int>(); gp.gb_beg = c->d_gb_beg.as<int>(); gp.gb_end = c->d_gb_end.as<int>();
    gp.ent_node = c->d_ent_node.as<int>(); gp.g_pack = c->d_g_pack.as<double>(); gp.gb_k0 = c->d_gb_k0.as<int>();
    gp.atom_coff = c->d_atom_coff.as<long long>(); gp.atom_npj = c->d_atom_npj.as<int>();
    gp.C = dC; gp.ldc = ldc;
    dim3 gg(c->n_gather_blocks, (nvec + 16 * kGatherNT - 1) / (16 * kGatherNT));
    for (int part = 0; part < (c->proj_complex ? 2 : 1); ++part) {
        if (part == 1) { gp.g_pack = c->d_g_pack_im.as<double>(); gp.C = dC2; }
        ProfScope ps(c, CSF_KIND_PGATHER);
        if (c->npjp <= 24) proj_gather_kernel<3, double><<<gg, 256, 0, c->stream>>>(gp);
        else proj_gather_kernel<4, double><<<gg, 256, 0, c->stream>>>(gp);
        CSF_CUDA(c, cudaGetLastError());
        c->launches += 1;
    }
    DeltaPlainParams dp{};
    dp.C = reinterpret_cast<const double2*>(dC); dp.C2 = c->proj_complex ? reinterpret_cast<const double2*>(dC2) : nullptr;
    dp.D = dD; dp.ldc = ldc; dp.nvec = nvec; dp.fr = fr; dp.fi = fi;
    dp.atom_coff = c->d_atom_coff.as<long long>(); dp.atom_npj = c->d_atom_npj.as<int>(); dp.atom_type = c->d_atom_type.as<int>();
    dp.delta = c->d_delta.as<double2>(); dp.delta_ptr = c->d_delta_ptr.as<long long>();
    { ProfScope ps(c, CSF_KIND_DELTA); delta_plain_kernel<<<dim3(c->natoms, (nvec + 31) / 32), 256, 0, c->stream>>>(dp); }
    CSF_CUDA(c, cudaGetLastError());
    ExpandPlainParams ep{};
    ep.D = dD; ep.ldc = ldc; ep.Y = dst; ep.ldy = ld_dst; ep.nvec = nvec; ep.mt = c->npjp <= 24 ? 3 : 4;
    ep.gb_atom = gp.gb_atom; ep.gb_beg = gp.gb_beg; ep.gb_end = gp.gb_end; ep.gb_k0 = gp.gb_k0; ep.ent_node = gp.ent_node;
    ep.g_pack = c->d_g_pack.as<double>(); ep.g_pack_im = c->d_g_pack_im.as<double>();
    ep.atom_coff = gp.atom_coff; ep.atom_npj = gp.atom_npj;
    {
        ProfScope ps(c, CSF_KIND_AUX);
        const dim3 eg(c->n_gather_blocks, (nvec + 31) / 32);
        if (c->proj_complex) expand_plain_kernel<true><<<eg, 256, 0, c->stream>>>(ep); else expand_plain_kernel<false><<<eg, 256, 0, c->stream>>>(ep);
    }
    CSF_CUDA(c, cudaGetLastError());
    c->launches += 2;
    return CSF_OK;
}

static int check_dense_args(csf_ctx* c, const void* dX, const void* dY, int64_t ld, int nvec, const void* d_work, size_t work_bytes, size_t need) {
    if (!dX || !dY) return fail(c, CSF_EINVAL, "NULL block pointer");
    if (dX == dY) return fail(c, CSF_EINVAL, "Y must not alias X");
    if (nvec < 0 || ld < nvec) return fail(c, CSF_EINVAL, "need 0 <= nvec <= ld");
    if (c->dense_nq == 0) return fail(c, CSF_ESTATE, "csf_set_potential_quadrature has not been called (it must follow csf_set_kpoint)");
    if (nvec > 0 && need > 0 && (!d_work || work_bytes < need)) return fail(c, CSF_EINVAL, "workspace too small");
    return CSF_OK;
}

int csf_apply_H_dense(csf_ctx* c, const csf_c128* dX, csf_c128* dY, int64_t ld, int nvec, void* d_work, size_t work_bytes) {
    CSF_GUARD_BEGIN
    if (!c) return CSF_EINVAL;
    // (one apply needs the coefficient buffers only; csf_dense_workspace_bytes also covers csf_filter_dense's block buffer)
    int rc = check_dense_args(c, dX, dY, ld, nvec, d_work, work_bytes, c->natoms > 0 ? 3 * coef_bytes(c, std::max(nvec, 0)) : 0);
    if (rc != CSF_OK || nvec == 0) return rc;
    CSF_CUDA(c, cudaSetDevice(c->device));
    rc = enqueue_zero(c, reinterpret_cast<double*>(dY), ld, nvec);
    if (rc != CSF_OK) return rc;
    char* coef = static_cast<char*>(d_work);
    return enqueue_dense_step(c, reinterpret_cast<const double2*>(dX), ld, reinterpret_cast<double*>(dY), ld, nvec, 1.0, 0, 0.0, coef);
    CSF_GUARD_END(c)
}

int csf_filter_dense(csf_ctx* c, const csf_c128* dX, csf_c128* dY, int64_t ld, int nvec, int degree, double a, double b, void* d_work, size_t work_bytes) {
    CSF_GUARD_BEGIN
    if (!c) return CSF_EINVAL;
    if (degree < 0) return fail(c, CSF_EINVAL, "degree < 0");
    if (!(a < b)) return fail(c, CSF_EINVAL, "need a < b");
    size_t need = 0; csf_dense_workspace_bytes(c, std::max(nvec, 0), &need);
    int rc = check_dense_args(c, dX, dY, ld, nvec, d_work, work_bytes, degree >= 1 ? need : 0);
    if (rc != CSF_OK || nvec == 0) return rc;
    CSF_CUDA(c, cudaSetDevice(c->device));
    const long long rows = 2 * c->M;
    const double cc = 0.5 * (a + b), ee = 0.5 * (b - a);
    const double2* X = reinterpret_cast<const double2*>(dX);
    double* Y = reinterpret_cast<double*>(dY);
    if (degree == 0) {
        { ProfScope ps(c, CSF_KIND_AUX); rot_copy_kernel<<<c->sm_count * 8, 256, 0, c->stream>>>(X, ld, reinterpret_cast<double2*>(Y), ld, rows, nvec, 0); }
        CSF_CUDA(c, cudaGetLastError()); c->launches += 1;
        return CSF_OK;
    }
    // the accumulate form of csf_filter: W_k = i^(m-k) T_k(H~) X, W_{k+1} = W_{k-1} + (-2i/e)(Hhat - c) W_k, W_m = T_m(H~) X
    char* w = static_cast<char*>(d_work);
    double* Wk = reinterpret_cast<double*>(w);
    char* coef = w + block_bytes(c, nvec);
    const bool even_m = (degree % 2 == 0);
    double* buf0 = even_m ? Y : Wk;  const long long ld0 = even_m ? ld : nvec;
    double* buf1 = even_m ? Wk : Y;  const long long ld1 = even_m ? nvec : ld;
    if (degree >= 2) {
        { ProfScope ps(c, CSF_KIND_AUX); rot_copy_kernel<<<c->sm_count * 8, 256, 0, c->stream>>>(X, ld, reinterpret_cast<double2*>(buf0), ld0, rows, nvec, degree & 3); }
        CSF_CUDA(c, cudaGetLastError()); c->launches += 1;
    }
    rc = enqueue_zero(c, buf1, ld1, nvec); if (rc != CSF_OK) return rc;
    rc = enqueue_dense_step(c, X, ld, buf1, ld1, nvec, 1.0 / ee, (degree + 3) & 3, cc, coef);
    if (rc != CSF_OK) return rc;
    for (int k = 1; k < degree; ++k) {
        const bool odd = (k & 1);
        rc = enqueue_dense_step(c, reinterpret_cast<const double2*>(odd ? buf1 : buf0), odd ? ld1 : ld0, odd ? buf0 : buf1, odd ? ld0 : ld1, nvec, 2.0 / ee, 3, cc, coef);
        if (rc != CSF_OK) return rc;
    }
    return CSF_OK;
    CSF_GUARD_END(c)
}

}  // extern "C"
