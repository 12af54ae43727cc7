// csf_kernels.cuh — hand-written sm_100a kernels of the Chebyshev-filtered spinor H.X.
//
// One recurrence step is  dst += gamma (Hhat - c) src  with gamma = sc * i^rot  ("accumulate form":
// with W_k = i^(m-k) T_k(H~) X the three-term recurrence of PAPER.md eq.70 becomes
// W_{k+1} = W_{k-1} + (-2i/e)(Hhat - c) W_k, a pure accumulation into the buffer that holds W_{k-1};
// multiplying by a power of i is exact in binary floating point). Per step three kernels run:
//
//   proj_gather_kernel   C^a  = P~^aT src|supp(a)                     (eq.84 inner sum, a5)
//   delta_apply_kernel   C~^a = Delta^{gamma_a} C^a                   (eq.76, a6)
//   column_kernel        gather -> sum-factorised 1/2 K -> nodal 2x2 potential, shift and projector
//                        expansion on the nodes the cell owns -> scaled scatter-add   (a1-a4, a7, a8; csf_column.cuh)
//
// Data layout: multivector element (node I, spin s, vector v) = complex128 at [(2I+s)*ld + v]. The operator
// tables are real, so the real and imaginary parts are independent batch entries: a "lane" is one double of
// the (spin, vector, re/im) batch and the lanes of a warp cover contiguous 8-byte words of 64-byte row pieces.
// The projector contractions (a5, a7) are FP64 tensor-core tiles (mma.sync m8n8k4) with both operands stored in
// fragment order; rot_narrow_kernel / widen_kernel convert between complex128 and complex64 for CSF_FP32_INTERMEDIATE.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace csf {

constexpr int kTabN = 8;

// ---------------------------------------------------------------------------------------------------
// proj_gather_kernel (a5): C[atom][2 chi + s][v] += sum_{I in the block's entry range} P~_{I chi} src[(2I+s)][v]
// as FP64 tensor-core tiles (mma.sync m8n8k4): A = P~^T (8 projectors x 4 support rows), B = src (4 rows x 8 real
// lanes = 4 vectors), D (8 projectors x 4 complex vectors) accumulated over the entry range and RED-added into C.
// grid.x = gather blocks (atom, <= 256 entries), grid.y = chunks of 32 vectors; the 8 warps of a CTA are
// (spin, 8 vectors) and read the same P~ rows (L1), every src element is read exactly once per H apply.
// ---------------------------------------------------------------------------------------------------
struct GatherParams {
    const void* src; long long ld; int nvec;       // src: complex128 or complex64 block (template parameter T)
    const int* gb_atom; const int* gb_beg; const int* gb_end;   // gather blocks over the entry list
    const int* gb_k0;                                            // first k-step (4 entries) of the block in g_pack
    const int* ent_node; const double* g_pack;                   // P~^T in A-fragment order [k-step][MT][32]
    const long long* atom_coff; const int* atom_npj;
    double* C; long long ldc;
};

__device__ __forceinline__ void gather_dmma(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

constexpr int kGatherNT = 4;     // n-tiles (of 4 vectors) per warp

// MT projector tiles of 8 in g_pack (npjp <= 8 MT); the first MD of them go through DMMA, NX further projectors
// (8 MD .. 8 MD + NX - 1, e.g. 16 and 17 of 18) by plain FMAs, which saves a mostly empty tensor tile; T = real type of src
template <int MT, typename T, int MD = MT, int NX = 0>
__global__ void __launch_bounds__(256, 2) proj_gather_kernel(const __grid_constant__ GatherParams A) {
    const int wl = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int kk = wl & 3, rw = wl >> 2;
    const int spin = warp & 1;
    const int v0 = blockIdx.y * (16 * kGatherNT) + (warp >> 1) * (4 * kGatherNT);
    if (v0 >= A.nvec) return;
    const int atom = A.gb_atom[blockIdx.x];
    const int e0 = A.gb_beg[blockIdx.x], e1 = A.gb_end[blockIdx.x];
    const int npj = A.atom_npj[atom];
    double acc[MD][kGatherNT][2];
    double accx[NX > 0 ? NX : 1][kGatherNT];
#pragma unroll
    for (int m = 0; m < MD; ++m)
#pragma unroll
        for (int nt = 0; nt < kGatherNT; ++nt) { acc[m][nt][0] = 0.0; acc[m][nt][1] = 0.0; }
#pragma unroll
    for (int x = 0; x < (NX > 0 ? NX : 1); ++x)
#pragma unroll
        for (int nt = 0; nt < kGatherNT; ++nt) accx[x][nt] = 0.0;
    const T* sb = static_cast<const T*>(A.src) + ((long long)spin * A.ld + v0 + (rw >> 1)) * 2 + (rw & 1);
    const double* gp = A.g_pack + (long long)A.gb_k0[blockIdx.x] * (MT * 32) + wl;
    constexpr int NA = MD + (NX > 0 ? NX : 0);      // a[0..MD) = DMMA A fragments, a[MD..) = this thread's row of the extra projectors
    // the node index of a support row is needed before its src row can be requested: it is fetched one round (two k-steps)
    // ahead of the data, so that the data loads never wait for an index
    auto load_node = [&](int e) { const int er = e + kk; return __ldg(A.ent_node + (er < e1 ? er : e0)); };
    auto load_step = [&](int e, int ks, int node, double (&a)[NA], double (&b)[kGatherNT]) {
        const int er = e + kk;
        const bool ok = er < e1;
#pragma unroll
        for (int m = 0; m < MD; ++m) a[m] = (e < e1) ? __ldg(gp + ((long long)ks * MT + m) * 32) : 0.0;
#pragma unroll
        for (int x = 0; x < NX; ++x) a[MD + x] = (e < e1) ? __ldg(gp - wl + ((long long)ks * MT + MD) * 32 + x * 4 + kk) : 0.0;
        const T* xp = sb + (long long)node * A.ld * 4;
#pragma unroll
        for (int nt = 0; nt < kGatherNT; ++nt) b[nt] = (ok && v0 + nt * 4 + (rw >> 1) < A.nvec) ? (double)__ldg(xp + nt * 8) : 0.0;
    };
    // two k-steps are multiplied while the next two are in flight
    double a0[NA], b0[kGatherNT], a1[NA], b1[kGatherNT];
    int n2 = load_node(e0 + 8), n3 = load_node(e0 + 12);
    load_step(e0, 0, load_node(e0), a0, b0);
    load_step(e0 + 4, 1, load_node(e0 + 4), a1, b1);
    int ks = 0;
    for (int e = e0; e < e1; e += 8, ks += 2) {
        double a2[NA], b2[kGatherNT], a3[NA], b3[kGatherNT];
        const int m2 = n2, m3 = n3;
        n2 = load_node(e + 16); n3 = load_node(e + 20);
        load_step(e + 8, ks + 2, m2, a2, b2);
        load_step(e + 12, ks + 3, m3, a3, b3);
#pragma unroll
        for (int m = 0; m < MD; ++m)
#pragma unroll
            for (int nt = 0; nt < kGatherNT; ++nt) gather_dmma(acc[m][nt][0], acc[m][nt][1], a0[m], b0[nt]);
#pragma unroll
        for (int m = 0; m < MD; ++m)
#pragma unroll
            for (int nt = 0; nt < kGatherNT; ++nt) gather_dmma(acc[m][nt][0], acc[m][nt][1], a1[m], b1[nt]);
#pragma unroll
        for (int x = 0; x < NX; ++x)
#pragma unroll
            for (int nt = 0; nt < kGatherNT; ++nt) accx[x][nt] = fma(a0[MD + x], b0[nt], fma(a1[MD + x], b1[nt], accx[x][nt]));
#pragma unroll
        for (int m = 0; m < NA; ++m) { a0[m] = a2[m]; a1[m] = a3[m]; }
#pragma unroll
        for (int nt = 0; nt < kGatherNT; ++nt) { b0[nt] = b2[nt]; b1[nt] = b3[nt]; }
    }
    const long long coff = A.atom_coff[atom];
    // extra projectors: sum the four support rows of a k-step (lanes kk = 0..3), lane kk = 0 adds real lane rw of its vector
#pragma unroll
    for (int x = 0; x < NX; ++x)
#pragma unroll
        for (int nt = 0; nt < kGatherNT; ++nt) {
            double v = accx[x][nt];
            v += __shfl_xor_sync(0xffffffffu, v, 1); v += __shfl_xor_sync(0xffffffffu, v, 2);
            const int vv = v0 + nt * 4 + (rw >> 1);
            if (kk == 0 && 8 * MD + x < npj && vv < A.nvec) atomicAdd(A.C + ((coff + 2 * (8 * MD + x) + spin) * A.ldc + vv) * 2 + (rw & 1), v);
        }
#pragma unroll
    for (int m = 0; m < MD; ++m) {
        const int chi = m * 8 + rw;
        if (chi < npj) {
#pragma unroll
            for (int nt = 0; nt < kGatherNT; ++nt) {
                const int v = v0 + nt * 4 + kk;
                if (v < A.nvec) {
                    double* cp = A.C + ((coff + 2 * chi + spin) * A.ldc + v) * 2;
                    atomicAdd(cp, acc[m][nt][0]); atomicAdd(cp + 1, acc[m][nt][1]);
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// proj_gather_bulk_kernel (a5, complex128 blocks): the same contraction with the src rows staged in shared memory by bulk
// asynchronous copies (cp.async.bulk global -> shared, completing on an mbarrier): one 1 KB request per (support row, spin)
// = 64 vectors, 16 rows per stage, kGbStages stages per CTA and two CTAs per SM, i.e. ~200 KB of src in flight per SM
// against ~32 KB with register loads (the register kernel sat at 59 % of the HBM copy rate, latency-bound). The B fragments
// then come from shared memory; a row stride of 2 KB + 64 B puts the four rows of a fragment on two bank halves.
// ---------------------------------------------------------------------------------------------------
constexpr int kGbRows = 16;                       // support rows per stage (4 k-steps)
constexpr int kGbStages = 3;
// bytes of a staged row: both spins x 64 vectors of complex<T>, + a skew that spreads the four rows of a B fragment over the
// banks (complex128: 64 bytes = two bank halves of 64-byte pieces; complex64: 32 bytes = four quarters of 32-byte pieces)
template <typename T> __host__ __device__ constexpr int gb_row_bytes() { return 2 * 64 * 2 * (int)sizeof(T) + (sizeof(T) == 8 ? 64 : 32); }
template <typename T> __host__ __device__ constexpr size_t gb_smem() { return (size_t)kGbStages * kGbRows * gb_row_bytes<T>() + 64; }
constexpr int kGbRowBytes = gb_row_bytes<double>();
constexpr size_t kGbSmem = gb_smem<double>();

// T = real type of the block (double: complex128 rows; float: the complex64 blocks of CSF_FP32_INTERMEDIATE, converted when
// the B fragments are read; the accumulation stays FP64). Complex64 rows are copied up to an even vector count (the blocks
// have an even leading dimension, so the pad column exists; its values never reach a fragment).
template <int MT, int MD, int NX, typename T = double>
__global__ void __launch_bounds__(256, 2) proj_gather_bulk_kernel(const __grid_constant__ GatherParams A) {
    constexpr int RB = gb_row_bytes<T>(), SPB = 64 * 2 * (int)sizeof(T), EB = 2 * (int)sizeof(T);      // row, spin half, complex element
    extern __shared__ __align__(128) unsigned char gsm[];
    const unsigned mb0 = (unsigned)__cvta_generic_to_shared(gsm + (size_t)kGbStages * kGbRows * RB);      // full[s], empty[s]
    const int tid = threadIdx.x, wl = tid & 31, warp = tid >> 5;
    const int kk = wl & 3, rw = wl >> 2;
    const int spin = warp & 1;
    const int vc0 = blockIdx.y * 64;                                     // first vector of this CTA
    const int vloc = (warp >> 1) * (4 * kGatherNT);                      // this warp's first vector inside the chunk
    const int nv = min(64, A.nvec - vc0);                                // live vectors of the chunk
    const int atom = A.gb_atom[blockIdx.x];
    const int e0 = A.gb_beg[blockIdx.x], e1 = A.gb_end[blockIdx.x];
    const int npj = A.atom_npj[atom];
    if (tid == 0) {
        for (int s = 0; s < kGbStages; ++s) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb0 + 8 * s));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 8;" ::"r"(mb0 + 8 * (kGbStages + s)));
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int ngroups = (e1 - e0 + kGbRows - 1) / kGbRows;
    // one warp issues the copies of a stage: lane = (row, spin); warp w issues groups w, w + 8, ... and holds the node index of its
    // next group's row (a copy must not wait for an index load)
    int nodep; { const int en = e0 + warp * kGbRows + (wl >> 1); nodep = en < e1 ? __ldg(A.ent_node + en) : 0; }
    auto issue = [&](int g) {
        const int s = g % kGbStages;
        const int eg = e0 + g * kGbRows, rows_g = min(kGbRows, e1 - eg);
        if (g >= kGbStages) {                                           // every warp has consumed the group that was in this stage
            unsigned done = 0;
            while (!done) asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }" : "=r"(done) : "r"(mb0 + 8 * (kGbStages + s)), "r"((unsigned)((g / kGbStages - 1) & 1)) : "memory");
        }
        const int cpb = ((nv * EB + 15) / 16) * 16;                     // bytes per (row, spin) copy
        if (wl == 0) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb0 + 8 * s), "r"((unsigned)(rows_g * 2 * cpb)) : "memory");
        __syncwarp();
        const int row = wl >> 1, sp = wl & 1;
        const long long node = nodep;
        { const int en = eg + 8 * kGbRows + row; nodep = en < e1 ? __ldg(A.ent_node + en) : 0; }      // this warp's next group: g + 8
        if (row < rows_g) {
            const char* src = static_cast<const char*>(A.src) + ((2 * node + sp) * A.ld + vc0) * EB;
            const unsigned dst = (unsigned)__cvta_generic_to_shared(gsm + ((size_t)s * kGbRows + row) * RB + sp * SPB);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"((unsigned)cpb), "r"(mb0 + 8 * s) : "memory");
        }
    };
    // the copies of group g are issued by warp g mod 8: a bulk copy costs the issuing warp ~500 cycles, and a fixed issuing warp
    // falls behind by that much in every group and sets the pace of the CTA through the stage barriers
    for (int g = 0; g < kGbStages && g < ngroups; ++g)
        if (warp == (g & 7)) issue(g);
    double acc[MD][kGatherNT][2];
    double accx[NX > 0 ? NX : 1][kGatherNT];
#pragma unroll
    for (int m = 0; m < MD; ++m)
#pragma unroll
        for (int nt = 0; nt < kGatherNT; ++nt) { acc[m][nt][0] = 0.0; acc[m][nt][1] = 0.0; }
#pragma unroll
    for (int x = 0; x < (NX > 0 ? NX : 1); ++x)
#pragma unroll
        for (int nt = 0; nt < kGatherNT; ++nt) accx[x][nt] = 0.0;
    const double* gp = A.g_pack + (long long)A.gb_k0[blockIdx.x] * (MT * 32) + wl;
    constexpr int NA = MD + (NX > 0 ? NX : 0);
    for (int g = 0; g < ngroups; ++g) {
        const int s = g % kGbStages;
        const int eg = e0 + g * kGbRows;
        // P~^T fragments of the group's four k-steps (global / L2), requested before the wait
        double a[4][NA];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const bool on = eg + 4 * q < e1;
#pragma unroll
            for (int m = 0; m < MD; ++m) a[q][m] = on ? __ldg(gp + ((long long)(4 * g + q) * MT + m) * 32) : 0.0;
#pragma unroll
            for (int x = 0; x < NX; ++x) a[q][MD + x] = on ? __ldg(gp - wl + ((long long)(4 * g + q) * MT + MD) * 32 + x * 4 + kk) : 0.0;
        }
        {
            unsigned done = 0;
            while (!done) asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }" : "=r"(done) : "r"(mb0 + 8 * s), "r"((unsigned)((g / kGbStages) & 1)) : "memory");
        }
        const T* sb = reinterpret_cast<const T*>(gsm + (size_t)s * kGbRows * RB + spin * SPB) + (vloc + (rw >> 1)) * 2 + (rw & 1);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const bool ok = eg + 4 * q + kk < e1;
            double b[kGatherNT];
#pragma unroll
            for (int nt = 0; nt < kGatherNT; ++nt)
                b[nt] = (ok && vloc + nt * 4 + (rw >> 1) < nv) ? (double)sb[(size_t)(4 * q + kk) * (RB / (int)sizeof(T)) + nt * 8] : 0.0;
#pragma unroll
            for (int m = 0; m < MD; ++m)
#pragma unroll
                for (int nt = 0; nt < kGatherNT; ++nt) gather_dmma(acc[m][nt][0], acc[m][nt][1], a[q][m], b[nt]);
#pragma unroll
            for (int x = 0; x < NX; ++x)
#pragma unroll
                for (int nt = 0; nt < kGatherNT; ++nt) accx[x][nt] = fma(a[q][MD + x], b[nt], accx[x][nt]);
        }
        __syncwarp();
        if (wl == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mb0 + 8 * (kGbStages + s)) : "memory");
        if (warp == ((g + kGbStages) & 7) && g + kGbStages < ngroups) issue(g + kGbStages);
    }
    const long long coff = A.atom_coff[atom];
    const int v0 = vc0 + vloc;
#pragma unroll
    for (int x = 0; x < NX; ++x)
#pragma unroll
        for (int nt = 0; nt < kGatherNT; ++nt) {
            double v = accx[x][nt];
            v += __shfl_xor_sync(0xffffffffu, v, 1); v += __shfl_xor_sync(0xffffffffu, v, 2);
            const int vv = v0 + nt * 4 + (rw >> 1);
            if (kk == 0 && 8 * MD + x < npj && vv < A.nvec) atomicAdd(A.C + ((coff + 2 * (8 * MD + x) + spin) * A.ldc + vv) * 2 + (rw & 1), v);
        }
#pragma unroll
    for (int m = 0; m < MD; ++m) {
        const int chi = m * 8 + rw;
        if (chi < npj) {
#pragma unroll
            for (int nt = 0; nt < kGatherNT; ++nt) {
                const int v = v0 + nt * 4 + kk;
                if (v < A.nvec) {
                    double* cp = A.C + ((coff + 2 * chi + spin) * A.ldc + v) * 2;
                    atomicAdd(cp, acc[m][nt][0]); atomicAdd(cp + 1, acc[m][nt][1]);
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// delta_apply_kernel: Ct[a][r][v] = sum_q Delta_t[r][q] C[a][q][v], r, q = 2 chi + s  (eq.76)
// grid = (atoms, vector chunks of 32); thread = (row group, vector).
// ---------------------------------------------------------------------------------------------------
struct DeltaParams {
    // Ct is written in the fragment order the column kernel's DMMA B operand wants: for (atom, chunk of VPC vectors)
    // a block [KS][L/8][32] doubles, element (s, nt, lane = rw*4 + kk) = C~[2 (4s + kk) + spin][vector].{re, im} with the
    // real lane nt*8 + rw = spin*(L/2) + 2*(vector % VPC) + ri; rows chi >= n_pj stay zero (the buffer is cleared).
    const double2* C; double* Ct; long long ldc; int nvec;
    int lanes, ks, nchunks;
    double scale;                 // C~ is stored times this factor (1, or the step's sc for the warp-specialised column kernel)
    const long long* atom_coff; const int* atom_npj; const int* atom_type;
    const double2* delta; const long long* delta_ptr;
};

__global__ void __launch_bounds__(256) delta_apply_kernel(const __grid_constant__ DeltaParams A) {
    const int atom = blockIdx.x;
    const int v = blockIdx.y * 32 + (threadIdx.x & 31);
    const int nr = 2 * A.atom_npj[atom];
    const double2* D = A.delta + A.delta_ptr[A.atom_type[atom]];
    const long long base = A.atom_coff[atom];
    if (v >= A.nvec) return;
    for (int r = threadIdx.x >> 5; r < nr; r += 8) {
        double sr = 0.0, si = 0.0;
        for (int q = 0; q < nr; ++q) {
            const double2 d = __ldg(D + (long long)r * nr + q);
            const double2 c = A.C[(base + q) * A.ldc + v];
            sr = fma(d.x, c.x, sr); sr = fma(-d.y, c.y, sr);
            si = fma(d.x, c.y, si); si = fma(d.y, c.x, si);
        }
        const int chi = r >> 1, spin = r & 1, vpc = A.lanes / 4;
        const int dl = spin * (A.lanes / 2) + (v % vpc) * 2;
        double* o = A.Ct + ((((long long)atom * A.nchunks + v / vpc) * A.ks + (chi >> 2)) * (A.lanes / 8) + (dl >> 3)) * 32 + (dl & 7) * 4 + (chi & 3);
        o[0] = A.scale * sr; o[4] = A.scale * si;
    }
}

// dst = i^rot * src  (complex128 [rows][ld] -> [rows][ld]); used for W_0 = i^m X
__global__ void __launch_bounds__(256) rot_copy_kernel(const double2* __restrict__ src, long long ld, double2* __restrict__ dst,
                                                       long long ld_dst, long long rows, int nvec, int rot) {
    const long long total = rows * nvec;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long r = t / nvec; const int v = (int)(t % nvec);
        const double2 z = src[r * ld + v];
        double2 o;
        if (rot == 0) o = z;
        else if (rot == 1) o = make_double2(-z.y, z.x);
        else if (rot == 2) o = make_double2(-z.x, -z.y);
        else o = make_double2(z.y, -z.x);
        dst[r * ld_dst + v] = o;
    }
}

// complex128 [rows][ld] -> complex64 [rows][ld_dst], times i^rot (CSF_FP32_INTERMEDIATE: W_0 = i^m X)
__global__ void __launch_bounds__(256) rot_narrow_kernel(const double2* __restrict__ src, long long ld, float2* __restrict__ dst,
                                                         long long ld_dst, long long rows, int nvec, int rot) {
    const long long total = rows * nvec;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long r = t / nvec; const int v = (int)(t % nvec);
        const double2 z = src[r * ld + v];
        double2 o;
        if (rot == 0) o = z;
        else if (rot == 1) o = make_double2(-z.y, z.x);
        else if (rot == 2) o = make_double2(-z.x, -z.y);
        else o = make_double2(z.y, -z.x);
        dst[r * ld_dst + v] = make_float2((float)o.x, (float)o.y);
    }
}

// complex64 [rows][ld] -> complex128 [rows][ld_dst]
__global__ void __launch_bounds__(256) widen_kernel(const float2* __restrict__ src, long long ld, double2* __restrict__ dst,
                                                    long long ld_dst, long long rows, int nvec) {
    const long long total = rows * nvec;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long r = t / nvec; const int v = (int)(t % nvec);
        const float2 z = src[r * ld + v];
        dst[r * ld_dst + v] = make_double2((double)z.x, (double)z.y);
    }
}

// zero the nvec live columns of a [rows][ld] block
__global__ void __launch_bounds__(256) zero_kernel(double2* __restrict__ dst, long long rows, long long ld, int nvec) {
    const long long total = rows * nvec;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long r = t / nvec; const int v = (int)(t % nvec);
        dst[r * ld + v] = make_double2(0.0, 0.0);
    }
}

// ---------------------------------------------------------------------------------------------------
// FP64 peak probes (csf_probe_fp64_peak): register-resident dependent chains, no memory traffic.
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) probe_dfma_kernel(double* sink, int iters, double m) {
    double a0 = threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double c = 1e-9;
#pragma unroll 4
    for (int it = 0; it < iters; ++it) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 12345.678) sink[threadIdx.x] = s;
}

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(256) probe_dmma_kernel(double* sink, int iters, double m) {
    double d[8][2];
#pragma unroll
    for (int q = 0; q < 8; ++q) { d[q][0] = threadIdx.x + q; d[q][1] = threadIdx.x - q; }
    const double a = m * 1e-3, b = 1e-3 * (threadIdx.x & 3);
#pragma unroll 2
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < 8; ++q) dmma884(d[q][0], d[q][1], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 8; ++q) s += d[q][0] + d[q][1];
    if (s == 12345.678) sink[threadIdx.x] = s;
}

// even warps run the DFMA chains, odd warps the DMMA chains: do the two instruction kinds have separate execution units?
__global__ void __launch_bounds__(256) probe_mixed_kernel(double* sink, int iters, double m) {
    if (((threadIdx.x >> 5) & 1) == 0) {
        double a0 = threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
        const double c = 1e-9;
#pragma unroll 4
        for (int it = 0; it < iters; ++it) {
            a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
            a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
        }
        const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
        if (s == 12345.678) sink[threadIdx.x] = s;
    } else {
        double d[8][2];
#pragma unroll
        for (int q = 0; q < 8; ++q) { d[q][0] = threadIdx.x + q; d[q][1] = threadIdx.x - q; }
        const double a = m * 1e-3, b = 1e-3 * (threadIdx.x & 3);
#pragma unroll 2
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int q = 0; q < 8; ++q) dmma884(d[q][0], d[q][1], a, b);
        }
        double s = 0.0;
#pragma unroll
        for (int q = 0; q < 8; ++q) s += d[q][0] + d[q][1];
        if (s == 12345.678) sink[threadIdx.x] = s;
    }
}

}  // namespace csf
