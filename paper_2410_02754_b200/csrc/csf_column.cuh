// csf_column.cuh — the column kernel: one recurrence step  dst += gamma (Hhat - c) src  of PAPER.md eq.70/eq.84
// for one z-segment of a column of cells and L/4 spinor vectors per CTA.
//
// Paper steps fused here: a1 extraction X^(e) = R^(e) X with the M_D^{-1/2} scaling folded into the
// 1-D operators, a2 cell-level product with the sum-factorised 1/2 K^(e), a3 nodal 2x2 spin potential, a7 projector
// expansion P^a C~^a (FP64 tensor-core tiles, mma.sync m8n8k4 = DMMA; inputs staged by TMA), a4 assembly (RED.F64),
// a8 recurrence update (accumulate form, csf_kernels.cuh).
//
// Why a column and not a cell: the L2 <-> SM fabric of B200 is barely faster than HBM, so the (n/p)^3 re-read /
// re-add of the shared cell faces is real time. A CTA that marches through S cells of one (cx, cy) column keeps the
// shared z-face on chip: its x-y contracted planes a2, b2 stay in a ring of N = p+1 shared-memory planes (they are
// identical for the upper cell's bottom plane and the lower cell's top plane), and the partial sums of the top
// plane are carried in registers into the next cell. Loads, x-y work and REDs all drop by p/(p+1).
//
// Operator tables. With the Loewdin scaling the 1-D operators of direction d are (csf_tables.h)
//     A_d = (2/h_d^2) Ah,   B_d = diag(beta) - uh uh^T,   beta = 1/2 on the two shared end nodes, 1 inside,
// where Ah and uh depend on the order p only. Ah is symmetric and centro-symmetric, uh is (anti)symmetric, so only
// N^2/4 + N/2 + N/2 distinct numbers occur; the kernel reads each entry through its canonical index and the whole
// table set stays resident in uniform registers (sm_100 has no constant-bank operand for DFMA). The kernel computes
//     out / ax = Bz (By Ah u + rho_y Ah Bx u) + rho_z Ah (By Bx u),   ax = 2/h_x^2, rho_d = h_x^2 / h_d^2.
//
// Warp roles. Main threads = (q, lane): L lanes = (spin, vector, re/im) are independent real streams of the same
// operator (the tables are real); q indexes a plane.
//   phase A  thread holds the x-y plane u[j][i] of one new z-plane in registers:
//              a2 = By Ah u + rho_y Ah Bx u,  b2 = rho_z By Bx u  -> ring
//   phase B  thread j takes the z-lines (j, i): out = ax (Bz a2 + Ah b2) (+ X on owned nodes, + carry on k = 0),
//              RED.F64 into dst for k < p, out[p] becomes the carry.
// Two auxiliary warps build X, the nodal and nonlocal terms on the owned nodes of the cell, beside phase A:
//   - one thread issues two TMA loads (cp.async.bulk.tensor + mbarrier): the src rows of the owned nodes (both spins,
//     this CTA's vectors) land in X, their V, Bx, By, Bz in a small stage; Dirichlet faces and vectors >= nvec are
//     zero-filled by the out-of-bounds rule;
//   - X = (V + B.sigma - c) X in place, thread = (node, vector) with both spins in registers;
//   - X += sum_a P~^a C~^a per (cell, atom) sub-pair as DMMA tiles (8 support rows x 8 lanes x 4 projectors); both
//     operands are stored in fragment order, so each fragment is one coalesced 256-byte load. Each warp owns one half
//     of the rows. The tensor pipe works while the FP64 pipe does phase A.
// X and the stage are double-buffered: the auxiliary warps work one cell ahead and meet the main warps at named
// barriers ("X[b] full" / "X[b] free", bar.arrive + bar.sync). The real type T is double (complex128 blocks) or float
// (CSF_FP32_INTERMEDIATE: complex64 blocks, FP32 cell arithmetic; the DMMA tiles and their operands stay FP64).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>

namespace csf {

constexpr int kColTab = 8;
// X / potential-stage buffers: the expansion warps run one cell ahead. (A third buffer fits at order 5 with 2 CTAs/SM
// but measured slower, 47.1 against 44.7 ms: it takes the shared-memory carve-out to 228 KB and leaves ~28 KB of L1.)
constexpr int kColXBuf = 2;
// expansion warps per CTA (each owns an equal share of the owned-node rows of X): 3 for the FP64 kernel of order 5 on
// periodic cubic meshes (measured: 48.9 -> 44.1 ms at config 3), 2 everywhere else (3 costs a CTA per SM at order 4, and
// the general order-5 kernel of config 2 measured 49.7 against 43.4 ms with 3). Wide kernels (32 lanes) of order 5 in
// FP64: CSF_WIDE_AUXW (the expansion work per CTA doubles with the lane count).
#ifndef CSF_WIDE_AUXW
#define CSF_WIDE_AUXW 4
#endif
#ifndef CSF_PREFB_MIN
#define CSF_PREFB_MIN 168
#endif
constexpr int kColMaxAuxWarps = 6;
constexpr int col_aux_warps(int p, bool f32, int mode, int lanes = 16) {
    if (lanes == 32) return (p == 5 && !f32) ? CSF_WIDE_AUXW : (p == 4 ? 3 : 2);
    return (p == 5 && !f32 && mode == 2) ? 3 : 2;
}
// first owned-node row of expansion warp r of nq (r = nq: one past the end); giving the warp that shares its SM
// sub-partition with two main warps a smaller share measured slower
__host__ __device__ constexpr int col_aux_row0(int nodes, int nq, int r) {
    const int split = (nodes + nq - 1) / nq;
    return r * split < nodes ? r * split : nodes;
}

// Fused projector gather (csf_filter on half-blocks, FP64, order 5, 8 vectors per CTA): two extra warps of the column kernel
// compute C = P~^T W for ANOTHER block of vectors (the half-block whose column step comes next) while the main warps work on
// this one. The gather is HBM-bound and the column step latency-bound, so the two share an SM at little cost to either.
// Tasks = (gather block of <= 256 support rows of one atom) x (chunk of kCgVec vectors), chunk fastest; CTA b takes tasks
// b, b + gridDim.x, ...
struct ColGather {
    const double* src; long long ld; int nvec;                  // complex128 block [2M][ld], nvec live vectors
    const int* gb_atom; const int* gb_beg; const int* gb_end;   // gather blocks over the entry list (as GatherParams)
    const int* gb_k0;                                            // first k-step (4 entries) of the block in g_pack
    const int* ent_node; const double* g_pack;                   // P~^T in A-fragment order [k-step][3][32]
    const long long* atom_coff; const int* atom_npj;
    double* C; long long ldc;                                    // [crows][ldc] complex128, cleared by the host, RED-added here
    int ntasks, nvc;                                             // tasks in all, vector chunks per gather block
};

struct ColParams {
    // TMA descriptors (cuTensorMapEncodeTiled): src viewed as [nfz][nfy][2 nfx rows][2 nvec doubles], box = the owned
    // nodes of one cell x L/2 doubles per spin row; vb viewed as [nfz][nfy][4 nfx doubles], box = one cell's owned nodes
    alignas(64) CUtensorMap tm_src;
    alignas(64) CUtensorMap tm_vb;
    double Ah[kColTab][kColTab];         // h-independent Loewdin-scaled 1-D stiffness (times 1/2), see above
    double uh[kColTab];                  // rank-one part of the 1-D mass
    float Ahf[kColTab][kColTab];         // the same tables rounded to FP32 (CSF_FP32_INTERMEDIATE)
    float uhf[kColTab];
    double ax, rho_y, rho_z;             // 2/h_x^2, h_x^2/h_y^2, h_x^2/h_z^2
    const void* src; void* dst;          // real type T = double (complex128 blocks) or float (complex64 blocks)
    int rs, rd;                          // reals per node in src / dst (4 * ld)
    int nvec;
    int ncx, ncy, ncz, nfx, nfy, nfz, bcx, bcy, bcz;
    const int* col_order; int ncols;     // traversal order of the (cx, cy) columns (8x8 tiles)
    int seg_len, nseg;                   // cells per z-segment, segments per column
    int chunk_group, nchunks;            // vector chunks of one column scheduled back to back; total chunks
    const double* vb;                    // [M][4] = V, Bx, By, Bz at the nodes
    double shift, sc; int rot;           // gamma = sc * i^rot, c = shift
    // projector expansion: (cell, atom) pairs, entries sorted by local owned index
    const int* sub_ptr;                  // [2 ncells + 1] sub-pairs (cell, atom, half of the owned-node range)
    const int4* sub_desc;                // [nsub] {atom, first tile in a_pack, entry begin, entry end}
    const double* a_pack;                // [ntiles][KS][32] P~ in DMMA A-fragment order (lane = row*4 + k), zero padded
    const int* ent_loc;                  // [nent] local owned index (lz*p + ly)*p + lx
    const double* Ct;                    // C~ in B-fragment order: [atom][chunk][KS][L/8][32] (DeltaParams)
    int npjp;
    long long* prof;                     // WS_PROF builds of csf_colws.cuh: per (CTA, warp) cycle counters
    ColGather g;                         // kernels with gather warps (GW > 0) only; ntasks = 0: nothing to gather
};

__device__ __forceinline__ double col_flip(double x, unsigned mask) {
    return __hiloint2double(__double2hiint(x) ^ (int)mask, __double2loint(x));
}
__device__ __forceinline__ float col_flip(float x, unsigned mask) { return __int_as_float(__float_as_int(x) ^ (int)mask); }

// fire-and-forget reduction (REDG): plain atomicAdd compiles to ATOMG with a discarded result inside this kernel
__device__ __forceinline__ void col_red(double* p, double v) { asm volatile("red.relaxed.gpu.global.add.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory"); }
__device__ __forceinline__ void col_red(float* p, float v) { asm volatile("red.relaxed.gpu.global.add.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory"); }

template <typename T> struct ColVec2;
template <> struct ColVec2<double> { using type = double2; };
template <> struct ColVec2<float> { using type = float2; };

__device__ __forceinline__ int col_free_index(int f, int ncell, int p, int bc) {
    const int nfull = ncell * p;
    if (bc == 0) return f >= nfull ? f - nfull : f;
    return (f == 0 || f == nfull) ? -1 : f - 1;
}

__device__ __forceinline__ void col_dmma(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// named barriers: 1 = main threads only; 2 + b = "X buffer b is full" (expansion warps arrive, main threads wait);
// 4 + b = "X buffer b is free" (main threads arrive, expansion warps wait; only when an expansion warp issues the TMA)
__device__ __forceinline__ void col_bar_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void col_bar_arrive(int id, int count) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory"); }

// gather warps (fused projector gather): each of the two warps (= spins) runs its own copy pipeline of kCgStages stages. A
// stage is one k-step: 4 support rows x kCgVec complex128 of the warp's spin (512 bytes each) and the k-step's P~^T fragments
// (the first 576 bytes of its 768 in g_pack: two DMMA tiles + the rows of projectors 16, 17). Laid out as
// [row 0][row 2][P~^T][row 1][row 3], the rows k = 0..3 of a B fragment sit on two bank halves (576 = 64 mod 128).
// Measured on the way here (config 3, cycles of a gather warp per k-step, 288 of them FP64-pipe time):
//  * the whole staging area must stay under ~16.7 KB: with more, the CTA no longer fits the 196 KB shared-memory
//    configuration, and the 228 KB one leaves the column step too little L1 (idle gather warps: 1617 against 1528 ms per block);
//  * P~^T fragments loaded into registers one k-step ahead arrive late, and so does a support row's node index loaded right
//    before its copy (the warp issues in order): fragments go through the pipeline, indices are fetched 32 rows at a time;
//  * cp.async.bulk costs the issuing warp ~500 cycles per k-step whatever the number of requests (1 x 4 lanes, 3 x 1 lane and
//    4 + 1 lanes all measured 530-640); plain 16-byte cp.async (LDGSTS, lane = 16-byte piece of a row) issues in ~400 and
//    makes a task 25 % shorter, but loads the LSU that the main warps depend on: 1853 against 1818 ms per block. Bulk copies stay.
#ifndef CSF_CG_STAGES
#define CSF_CG_STAGES 3
#endif
constexpr int kCgStages = CSF_CG_STAGES, kCgVec = 32;
constexpr int kCgRowBytes = kCgVec * 16;                                          // one spin of one support row
constexpr int kCgABytes = 2 * 256 + 64;                                           // P~^T of one k-step as far as it is read
constexpr int kCgStageBytes = 4 * kCgRowBytes + kCgABytes;
constexpr int kCgWarpBytes = kCgStages * kCgStageBytes;
constexpr size_t kCgBytes = (size_t)2 * kCgWarpBytes + 2 * kCgStages * 8;        // two warps + their full[s] mbarriers
__host__ __device__ constexpr int col_cg_row(int k) { return (k >> 1) * kCgRowBytes + ((k & 1) ? 2 * kCgRowBytes + kCgABytes : 0); }
constexpr int kCgAOff = 2 * kCgRowBytes;

// ---------------------------------------------------------------------------------------------------------------
// Gather role (a5 inside the column kernel): C[atom][2 chi + s][v] += sum_I P~_{I chi} src[(2I+s)][v] (eq.84 inner
// sum) for the task list of this CTA. Two warps = the two spins, each with its own pipeline; a warp holds 8 n-tiles of 4
// vectors. Support rows and P~^T fragments are staged in shared memory by cp.async.bulk (lanes 0-3 copy a row each, lane 4 the
// fragments, all completing on the stage's mbarrier), projectors 0-15 go through DMMA m8n8k4 tiles (A = P~^T 8 x 4 in
// fragment order, B = src 4 rows x 8 real lanes), 16 and 17 by plain FMAs — the arithmetic of
// proj_gather_bulk_kernel<3, 2, 2> (csf_kernels.cuh), which serves 18 projectors per atom.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void col_gather_role(const ColGather& G, unsigned char* gsm, int gw, int wl) {
    constexpr int MT = 3, MD = 2, NX = 2, NTG = kCgVec / 4;
    unsigned char* const wsm = gsm + (size_t)gw * kCgWarpBytes;
    const unsigned wsm_u = (unsigned)__cvta_generic_to_shared(wsm);
    const unsigned mb0 = (unsigned)__cvta_generic_to_shared(gsm + (size_t)2 * kCgWarpBytes) + gw * (kCgStages * 8);      // full[s] of this warp
    const int kk = wl & 3, rw = wl >> 2, spin = gw;
    if (wl == 0) {
#pragma unroll
        for (int s = 0; s < kCgStages; ++s) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb0 + 8 * s));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    int gbase = 0;                  // k-steps staged so far by this warp: stage and mbarrier phase continue across tasks
    for (int task = blockIdx.x; task < G.ntasks; task += gridDim.x) {
        const int gb = task / G.nvc, vc0 = (task % G.nvc) * kCgVec;
        const int nv = min(kCgVec, G.nvec - vc0);
        const int atom = __ldg(G.gb_atom + gb), e0 = __ldg(G.gb_beg + gb), e1 = __ldg(G.gb_end + gb);
        const int nks = (e1 - e0 + 3) / 4;
        const char* const srcb = reinterpret_cast<const char*>(G.src) + ((long long)spin * G.ld + vc0) * 16;
        const char* const gpb = reinterpret_cast<const char*>(G.g_pack + (long long)__ldg(G.gb_k0 + gb) * (MT * 32));
        // node indices of the support rows, 8 k-steps (32 rows) per coalesced load, two batches in registers: a copy must
        // not wait for its row's index (the warp issues in order, and one round trip to L2 per k-step is what bounds it then)
        auto load_idx = [&](int b) { const int e = e0 + 32 * b + wl; return e < e1 ? __ldg(G.ent_node + e) : 0; };
        int idx0 = load_idx(0), idx1 = load_idx(1);
        // stage k-step g of this task (called with g = 0, 1, 2, ... in order): lane k < 4 copies support row k (this warp's
        // spin), lane 4 the P~^T fragments; the warp has finished reading the stage (program order + the warp-wide shuffle)
        auto issue = [&](int g) {
            const int s = (gbase + g) % kCgStages;
            const int eg = e0 + 4 * g, rows_g = min(4, e1 - eg);
            const unsigned sbase = wsm_u + (unsigned)(s * kCgStageBytes);
            const int bt = g >> 3;
            if ((g & 7) == 0 && g > 0) { if (bt & 1) idx0 = load_idx(bt + 1); else idx1 = load_idx(bt + 1); }      // batch bt - 1 is used up
            const long long node = __shfl_sync(0xffffffffu, (bt & 1) ? idx1 : idx0, (g & 7) * 4 + (wl & 3));
            if (wl == 0) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb0 + 8 * s), "r"((unsigned)(rows_g * nv * 16 + kCgABytes)) : "memory");
            __syncwarp();
            if (wl < rows_g) {
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                             ::"r"(sbase + (unsigned)col_cg_row(wl)), "l"(srcb + 2 * node * G.ld * 16), "r"((unsigned)(nv * 16)), "r"(mb0 + 8 * s) : "memory");
            } else if (wl == 4) {
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                             ::"r"(sbase + (unsigned)kCgAOff), "l"(gpb + (long long)g * (MT * 256)), "r"((unsigned)kCgABytes), "r"(mb0 + 8 * s) : "memory");
            }
        };
        for (int g = 0; g < kCgStages && g < nks; ++g) issue(g);
        double acc[MD][NTG][2], accx[NX][NTG];
#pragma unroll
        for (int m = 0; m < MD; ++m)
#pragma unroll
            for (int nt = 0; nt < NTG; ++nt) { acc[m][nt][0] = 0.0; acc[m][nt][1] = 0.0; }
#pragma unroll
        for (int x = 0; x < NX; ++x)
#pragma unroll
            for (int nt = 0; nt < NTG; ++nt) accx[x][nt] = 0.0;
        for (int g = 0; g < nks; ++g) {
            {
                const int gi = gbase + g; unsigned done = 0;
                while (!done) asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }" : "=r"(done) : "r"(mb0 + 8 * (gi % kCgStages)), "r"((unsigned)((gi / kCgStages) & 1)) : "memory");
            }
            const unsigned char* st = wsm + ((gbase + g) % kCgStages) * kCgStageBytes;
            const bool ok = e0 + 4 * g + kk < e1;               // rows past the block's end were not copied: stale data
            const double* sb = reinterpret_cast<const double*>(st + col_cg_row(kk)) + rw;
            const double* sa = reinterpret_cast<const double*>(st + kCgAOff);
            double a[MD + NX], b[NTG];
#pragma unroll
            for (int m = 0; m < MD; ++m) a[m] = sa[m * 32 + wl];
#pragma unroll
            for (int x = 0; x < NX; ++x) a[MD + x] = sa[MD * 32 + x * 4 + kk];
#pragma unroll
            for (int nt = 0; nt < NTG; ++nt) b[nt] = (ok && nt * 4 + (rw >> 1) < nv) ? sb[nt * 8] : 0.0;
#pragma unroll
            for (int m = 0; m < MD; ++m)
#pragma unroll
                for (int nt = 0; nt < NTG; ++nt) col_dmma(acc[m][nt][0], acc[m][nt][1], a[m], b[nt]);
#pragma unroll
            for (int x = 0; x < NX; ++x)
#pragma unroll
                for (int nt = 0; nt < NTG; ++nt) accx[x][nt] = fma(a[MD + x], b[nt], accx[x][nt]);
            if (g + kCgStages < nks) issue(g + kCgStages);
        }
        gbase += nks;
        const long long coff = __ldg(G.atom_coff + atom);
        const int npj = __ldg(G.atom_npj + atom);
        // extra projectors: sum the four support rows of a k-step (lanes kk = 0..3), lane kk = 0 adds real lane rw of its vector
#pragma unroll
        for (int x = 0; x < NX; ++x)
#pragma unroll
            for (int nt = 0; nt < NTG; ++nt) {
                double v = accx[x][nt];
                v += __shfl_xor_sync(0xffffffffu, v, 1); v += __shfl_xor_sync(0xffffffffu, v, 2);
                const int vv = vc0 + nt * 4 + (rw >> 1);
                if (kk == 0 && 8 * MD + x < npj && vv < G.nvec) col_red(G.C + ((coff + 2 * (8 * MD + x) + spin) * G.ldc + vv) * 2 + (rw & 1), v);
            }
#pragma unroll
        for (int m = 0; m < MD; ++m) {
            const int chi = m * 8 + rw;
            if (chi < npj) {
#pragma unroll
                for (int nt = 0; nt < NTG; ++nt) {
                    const int v = vc0 + nt * 4 + kk;
                    if (v < G.nvec) {
                        double* cp = G.C + ((coff + 2 * chi + spin) * G.ldc + v) * 2;
                        col_red(cp, acc[m][nt][0]); col_red(cp + 1, acc[m][nt][1]);
                    }
                }
            }
        }
    }
}

// canonical representative of (i, j) under transposition and the centro flip (i, j) -> (N-1-i, N-1-j)
template <int N> __host__ __device__ constexpr int col_canon(int i, int j) {
    int best = i * kColTab + j, c = j * kColTab + i;
    if (c < best) best = c;
    c = (N - 1 - i) * kColTab + (N - 1 - j); if (c < best) best = c;
    c = (N - 1 - j) * kColTab + (N - 1 - i); if (c < best) best = c;
    return best;
}

// Who issues the TMA loads of a cell: a main thread right after phase B has released the buffer, so that the expansion
// warps find their data waiting (orders >= 5: config 3 44.0 -> 40.9 ms), or the first expansion warp itself after a
// "buffer free" barrier (orders <= 4, where a cell is short and the extra work of the main thread costs more than the
// exposed TMA latency: config 4 44.9 against 45.5 ms). The wide kernel of order 4 (8 vectors per CTA, a cell takes twice
// as long) is on the main-thread side again: config 4 44.3 -> 39.8 ms, config 1 0.52 -> 0.47 ms per launch.
__host__ __device__ constexpr bool col_main_tma(int p, int lanes = 16) { return p >= 5 || (p == 4 && lanes == 32); }

// register cap per thread: what the CTAs/SM allowed by shared memory leave (orders 4, 5; other orders uncapped).
// L = 16: order 4 runs 3 CTAs/SM (FP32: 4), order 5 two (FP32: 3).
__host__ __device__ constexpr int col_maxreg(int p, bool f32, int lanes, int auxw) {
    if (p < 4 || p > 5) return 255;
    // The register file is per SM sub-partition (16384 registers): w warps per SM sit ceil(w / 4) per sub-partition.
    // 32 lanes, order 5: 6 main warps + auxw in one CTA/SM (FP64; up to 8 warps sit 2 per sub-partition, up to 12 sit 3) or
    // two CTAs of 8 warps (FP32); order 4: two CTAs of 5 + 3 warps.
    if (lanes == 32) return p == 4 ? 128 : (f32 ? 128 : (auxw <= 2 ? 224 : 168));
    return f32 ? (p == 4 ? 96 : 128) : (p == 4 ? 128 : 168);
}

template <typename T, int P, int L, int AUXW = 2, int GW = 0> struct ColCfg {
    static constexpr int N = P + 1;
    static constexpr int NTM = (N * L + 31) / 32 * 32;               // main threads
    static constexpr int NAUX = 32 * AUXW;                           // auxiliary (expansion) threads
    static constexpr int NTB = NTM + NAUX;                           // threads of the column step (named-barrier counts)
    static constexpr int NT = NTB + 32 * GW;                         // threads per CTA (+ gather warps, highest warp ids)
    static constexpr int PLANE = N * N * L;                          // reals per ring plane and field
    static constexpr int EPLANE = P * P * L;
    static constexpr int VCELL = P * P * P * 4;                      // V, Bx, By, Bz of the owned nodes of one cell
    // a2 ring, b2 ring, X (nodal + nonlocal terms on the owned nodes of the current cell), staged potential, mbarrier
    static constexpr size_t XOFF = ((size_t)2 * N * PLANE * sizeof(T) + 127) / 128 * 128;
    static constexpr size_t XBYTES = ((size_t)P * EPLANE * sizeof(T) + 127) / 128 * 128;          // one X buffer
    static constexpr size_t VBYTES = ((size_t)VCELL * sizeof(double) + 127) / 128 * 128;          // one potential stage
    static constexpr size_t VOFF = XOFF + kColXBuf * XBYTES;          // X and the stage are multi-buffered (cell t uses t % kColXBuf)
    static constexpr size_t MOFF = VOFF + kColXBuf * VBYTES;
    static constexpr size_t GOFF = (MOFF + 32 + 127) / 128 * 128;    // gather stages (GW > 0)
    static constexpr size_t SMEM = GW > 0 ? GOFF + kCgBytes : MOFF + 32;
};

// MODE 2: every node of the mesh is unconstrained (all directions periodic), nvec is a multiple of L/4 and the cells
// are cubes (rho_y = rho_z = 1), so no load, store or RED needs a predicate and no rho multiply is issued.
template <typename T, int P, int KS, int MODE, int L, int AUXW = col_aux_warps(P, sizeof(T) == 4, MODE, L), int GW = 0>
__global__ void __launch_bounds__(ColCfg<T, P, L, AUXW, GW>::NT) __maxnreg__(col_maxreg(P, sizeof(T) == 4, L, AUXW)) column_kernel(const __grid_constant__ ColParams A) {
    using Cfg = ColCfg<T, P, L, AUXW, GW>;
    constexpr int kColAuxWarps = AUXW, kColAux = Cfg::NAUX;
    constexpr bool kMainTma = col_main_tma(P, L), kPot2 = P >= 5;
    using T2 = typename ColVec2<T>::type;
    constexpr bool kWarpPlane = L % 32 == 0;      // a main warp holds exactly one plane
    constexpr bool FAST = MODE >= 1;      // x, y periodic and all lanes live: no per-access predicate
    constexpr bool ZISO = MODE == 2;      // z periodic too and cubic cells: no z check, no rho multiply
    constexpr int N = Cfg::N, NTM = Cfg::NTM, VPC = L / 4;        // VPC vectors per CTA
    constexpr int PLANE = Cfg::PLANE, EPLANE = Cfg::EPLANE;
    extern __shared__ __align__(128) unsigned char smem[];
    T* R1 = reinterpret_cast<T*>(smem);
    T* R2 = R1 + N * PLANE;
    char* const xbase = reinterpret_cast<char*>(smem) + Cfg::XOFF;
    char* const vbase = reinterpret_cast<char*>(smem) + Cfg::VOFF;
    const unsigned mbar0 = (unsigned)__cvta_generic_to_shared(reinterpret_cast<char*>(smem) + Cfg::MOFF);

    constexpr bool F32 = sizeof(T) == 4;
#define TAB_A(k) (F32 ? (T)(&A.Ahf[0][0])[k] : (T)(&A.Ah[0][0])[k])
#define TAB_U(k) (F32 ? (T)A.uhf[k] : (T)A.uh[k])
#define AH(i, j) TAB_A(col_canon<N>(i, j))
#define UH(i) (((P & 1) && (i) > N - 1 - (i)) ? -TAB_U(N - 1 - (i)) : TAB_U((i) < N - 1 - (i) ? (i) : N - 1 - (i)))
#define BETA(i) (((i) == 0 || (i) == P) ? (T)0.5 : (T)1.0)

    // ---- which (column, segment, vector chunk)
    int r = blockIdx.x;
    const int cg = r % A.chunk_group; r /= A.chunk_group;
    const int cidx = r % A.ncols; r /= A.ncols;
    const int seg = r % A.nseg; r /= A.nseg;
    const int chunk = r * A.chunk_group + cg;
    const bool live = chunk < A.nchunks;
    if constexpr (GW == 0) { if (!live) return; }
    else {
        // gather warps (the LOWEST warp ids: the scheduler favours high ids, which belong to the main warps; with 4 expansion
        // warps next, warps 0, 1 land on the SM sub-partitions that carry one main warp) work on their own task list, also in
        // a CTA that has no column work
        const int gwarp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
        if (gwarp < GW) { col_gather_role(A.g, smem + Cfg::GOFF, gwarp, (int)(threadIdx.x & 31)); return; }
        if (!live) return;
    }
    const int col = A.col_order[cidx];
    const int cx = col % A.ncx, cy = col / A.ncx;
    const int cz0 = seg * A.seg_len;
    const int S = min(A.seg_len, A.ncz - cz0);
    const int tid = (int)threadIdx.x - 32 * GW;          // thread index among the threads of the column step
    const int plane_nodes = A.nfx * A.nfy;

    if (tid == 0) {
#pragma unroll
        for (int b = 0; b < kColXBuf; ++b) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mbar0 + 8 * b));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if constexpr (GW == 0) __syncthreads(); else col_bar_sync(0, Cfg::NTB);

    // warp-uniform role (broadcast from lane 0 so that the compiler knows the branch does not split a warp)
    const int warp_id = __shfl_sync(0xffffffffu, tid >> 5, 0);
    // the expansion warps take the LOW warp ids: the scheduler favours high warp ids, and the main warps carry the
    // FP64 work, while the expansion warps mostly wait
    if (warp_id < kColAuxWarps) {
        // ============================================================== auxiliary warps
        // Warp aw owns the owned-node range [aw * XSPLIT, (aw + 1) * XSPLIT) of X, so the two warps never touch the
        // same row and need no barrier between them. Its sub-pairs (cell, atom, range) come from the host.
        const int aw = warp_id, wl = tid & 31;
        const int kk = wl & 3, rw = wl >> 2;
        constexpr int TMAX = (P * P * P + 7) / 8, TCH = TMAX < 5 ? TMAX : ((L == 32 && col_maxreg(P, sizeof(T) == 4, L, AUXW) <= 128) ? 3 : 5);   // wide kernels capped at 128 registers: fewer tiles in flight
        constexpr bool kPrefB = col_maxreg(P, sizeof(T) == 4, L, AUXW) > CSF_PREFB_MIN;
        const int xr0 = col_aux_row0(P * P * P, kColAuxWarps, aw), xr1 = col_aux_row0(P * P * P, kColAuxWarps, aw + 1);
        auto load_b = [&](const int4& ds, double (&bb)[KS][L / 8]) {
            const double* cb = A.Ct + ((long long)ds.x * A.nchunks + chunk) * (KS * (L / 8) * 32) + wl;
#pragma unroll
            for (int s = 0; s < KS; ++s)
#pragma unroll
                for (int nt = 0; nt < L / 8; ++nt) bb[s][nt] = __ldg(cb + (s * (L / 8) + nt) * 32);
        };
        for (int t = 0; t < S; ++t) {
            const int xb = t % kColXBuf;
            T* X = reinterpret_cast<T*>(xbase + xb * Cfg::XBYTES);
            double* VS = reinterpret_cast<double*>(vbase + xb * Cfg::VBYTES);
            const unsigned mbar = mbar0 + 8 * xb;
            // the first sub-pair's descriptor and C~ fragments do not depend on X: fetch them before any waiting
            int sp0 = 0, sp1 = 0;
            int4 ds = make_int4(0, 0, 0, 0);           // {atom, first tile in a_pack, entry begin, entry end}
            double b[KS][L / 8];
            if (A.sub_ptr != nullptr) {
                const int cell = cx + A.ncx * (cy + A.ncy * (cz0 + t));
                sp0 = A.sub_ptr[cell * kColAuxWarps + aw]; sp1 = A.sub_ptr[cell * kColAuxWarps + aw + 1];
                if (sp0 < sp1) { ds = __ldg(A.sub_desc + sp0); load_b(ds, b); }
            }
            if constexpr (!kMainTma) {
                if (t >= kColXBuf) col_bar_sync(4 + xb, Cfg::NTB);    // phase B(t - kColXBuf) has consumed this X buffer
                if (aw == 0 && wl == 0) {
                    const int bx0 = cx * P - (A.bcx == 0 ? 0 : 1), by0 = cy * P - (A.bcy == 0 ? 0 : 1), bz0 = (cz0 + t) * P - (A.bcz == 0 ? 0 : 1);
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"((unsigned)(P * EPLANE * sizeof(T) + Cfg::VCELL * sizeof(double))) : "memory");
                    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                                 ::"r"((unsigned)__cvta_generic_to_shared(X)), "l"(&A.tm_src), "r"(chunk * VPC * 2), "r"(bx0 * 2), "r"(by0), "r"(bz0), "r"(mbar) : "memory");
                    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                                 ::"r"((unsigned)__cvta_generic_to_shared(VS)), "l"(&A.tm_vb), "r"(bx0 * 4), "r"(by0), "r"(bz0), "r"(mbar) : "memory");
                }
            }
            // the TMA loads of cell t have landed
            {
                unsigned done = 0;
                while (true) {
                    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }" : "=r"(done) : "r"(mbar), "r"((unsigned)((t / kColXBuf) & 1)) : "memory");
                    if (done) break;
                    if constexpr (kMainTma) __nanosleep(200);       // the buffer is still in use by phase B: stay out of the main warps' way
                }
            }
            // X = (V + B.sigma - c) X in place on this warp's rows: thread = (node, vector), both spins and re/im in
            // registers, so the 2x2 spin block needs no exchange between threads; PW tasks per pass (independent chains).
            // (Swapping the spin halves of neighbouring nodes would remove the 2-way bank conflict of these accesses;
            // measured slower: the selects cost more than the conflicts.)
            {
                constexpr int PW = kPot2 ? 2 : 1;
                const int ntask = (xr1 - xr0) * VPC;
                for (int task0 = wl; task0 < ntask; task0 += 32 * PW) {
                    T2* xu[PW]; T2 uu[PW], ud[PW]; double2 v01[PW], v23[PW]; bool on[PW];
#pragma unroll
                    for (int w = 0; w < PW; ++w) {
                        const int task = task0 + 32 * w;
                        on[w] = PW == 1 || task < ntask;
                        const int loc = on[w] ? xr0 + task / VPC : xr0, vl = task % VPC;
                        xu[w] = reinterpret_cast<T2*>(X + loc * L) + vl;
                        uu[w] = xu[w][0]; ud[w] = xu[w][L / 4];
                        v01[w] = reinterpret_cast<const double2*>(VS)[2 * loc]; v23[w] = reinterpret_cast<const double2*>(VS)[2 * loc + 1];
                    }
#pragma unroll
                    for (int w = 0; w < PW; ++w) {
                        const T vv = (T)(v01[w].x - A.shift), bx = (T)v01[w].y, by = (T)v23[w].x, bz = (T)v23[w].y;
                        T2 ou, od;
                        ou.x = fma(vv + bz, uu[w].x, fma(bx, ud[w].x, by * ud[w].y));
                        ou.y = fma(vv + bz, uu[w].y, fma(bx, ud[w].y, -by * ud[w].x));
                        od.x = fma(vv - bz, ud[w].x, fma(bx, uu[w].x, -by * uu[w].y));
                        od.y = fma(vv - bz, ud[w].y, fma(bx, uu[w].y, by * uu[w].x));
                        if (on[w]) { xu[w][0] = ou; xu[w][L / 4] = od; }
                    }
                }
            }
            __syncwarp();
            {
                for (int sp = sp0; sp < sp1; ++sp) {
                    // A fragments of up to TCH tiles at once (one exposed round trip), next sub-pair's B meanwhile
                    const int e0 = ds.z, e1 = ds.w;
                    // (kernels capped at 128 registers prefetch the next descriptor only: its C~ fragments are requested
                    // together with its first P~ tiles, which is one exposed round trip either way, and 40 registers less)
                    int4 dn = ds; double bn[kPrefB ? KS : 1][kPrefB ? L / 8 : 1];
                    if (sp + 1 < sp1) { dn = __ldg(A.sub_desc + sp + 1); if constexpr (kPrefB) load_b(dn, bn); }
                    for (int eb = e0; eb < e1; eb += 8 * TCH) {
                        double a[TCH][KS]; int loc[TCH];
#pragma unroll
                        for (int tl = 0; tl < TCH; ++tl) {
                            const int erow = eb + tl * 8 + rw;
                            const bool vd = erow < e1, tv = eb + tl * 8 < e1;
                            const double* ap = A.a_pack + ((long long)(ds.y + ((eb - e0) >> 3) + (tv ? tl : 0)) * KS) * 32 + wl;
#pragma unroll
                            for (int s = 0; s < KS; ++s) a[tl][s] = tv ? __ldg(ap + s * 32) : 0.0;
                            loc[tl] = vd ? __ldg(A.ent_loc + erow) : -1;
                        }
#pragma unroll
                        for (int tl = 0; tl < TCH; ++tl) {
                            if (eb + tl * 8 < e1) {
                                double c[L / 8][2];
#pragma unroll
                                for (int nt = 0; nt < L / 8; ++nt) { c[nt][0] = 0.0; c[nt][1] = 0.0; }
#pragma unroll
                                for (int s = 0; s < KS; ++s)
#pragma unroll
                                    for (int nt = 0; nt < L / 8; ++nt) col_dmma(c[nt][0], c[nt][1], a[tl][s], b[s][nt]);
                                if (loc[tl] >= 0) {
                                    T2* ep = reinterpret_cast<T2*>(X + loc[tl] * L + 2 * kk);
#pragma unroll
                                    for (int nt = 0; nt < L / 8; ++nt) { T2 v = ep[4 * nt]; v.x += (T)c[nt][0]; v.y += (T)c[nt][1]; ep[4 * nt] = v; }
                                }
                            }
                        }
                    }
                    __syncwarp();          // the next sub-pair of this warp may touch the same rows from other lanes
                    if (sp + 1 < sp1) {
                        ds = dn;
                        if constexpr (kPrefB) {
#pragma unroll
                            for (int s = 0; s < KS; ++s)
#pragma unroll
                                for (int nt = 0; nt < L / 8; ++nt) b[s][nt] = bn[kPrefB ? s : 0][kPrefB ? nt : 0];
                        } else load_b(ds, b);
                    }
                }
            }
            __threadfence_block();
            col_bar_arrive(2 + xb, Cfg::NTB);                     // X(t) is complete
        }
        return;
    }

    // ================================================================== main warps
    const int mtid = tid - kColAux;
    const int lane = mtid % L, q = mtid / L;
    const int spin = lane / (L / 2), ri = lane & 1;
    const int vec = chunk * VPC + ((lane % (L / 2)) >> 1);
    const bool lane_on = FAST || vec < A.nvec;
    const bool q_on = q < N;

    // node offsets of the column's x / y indices (or -1 on a Dirichlet face). On a periodic mesh only the last index
    // of the last cell wraps, so the FAST kernel keeps two numbers per direction instead of the arrays.
    int xo_[FAST ? 1 : N], yo_[FAST ? 1 : N];
    const int x0f = cx * P, xPf = (cx == A.ncx - 1) ? 0 : cx * P + P;
    const int y0f = cy * P * A.nfx, yPf = (cy == A.ncy - 1) ? 0 : (cy * P + P) * A.nfx;
    if (!FAST) {
#pragma unroll
        for (int i = 0; i < N; ++i) {
            xo_[i] = col_free_index(cx * P + i, A.ncx, P, A.bcx);
            const int gy = col_free_index(cy * P + i, A.ncy, P, A.bcy);
            yo_[i] = gy < 0 ? -1 : gy * A.nfx;
        }
    }
#define XO(i) (FAST ? ((i) < P ? x0f + (i) : xPf) : xo_[FAST ? 0 : (i)])
#define YO(j) (FAST ? ((j) < P ? y0f + (j) * A.nfx : yPf) : yo_[FAST ? 0 : (j)])
    const T* sp = static_cast<const T*>(A.src) + ((long long)spin * (A.rs >> 2) + vec) * 2 + ri;
    const int slot_out = ri ^ (A.rot & 1);
    const unsigned sgn = (A.rot == 2 || (A.rot == 1 && ri == 1) || (A.rot == 3 && ri == 0)) ? 0x80000000u : 0u;
    T* dp = static_cast<T*>(A.dst) + ((long long)spin * (A.rd >> 2) + vec) * 2 + slot_out;
    const T scax = (T)(A.sc * A.ax);

    T u[N][N];
    T carry[N];
#pragma unroll
    for (int i = 0; i < N; ++i) carry[i] = (T)0;

    // plane of the segment handled by this thread in iteration t (segment-local plane index g), or -1
    auto plane_of = [&](int t) -> int {
        if (!q_on) return -1;
        if (t == 0) return q;
        const int rr = (q + t) % N;
        return rr < P ? t * P + rr + 1 : -1;
    };
    auto load_plane = [&](int g) {
        if (kWarpPlane && g < 0) return;
        const int gz = g < 0 ? (FAST ? 0 : -1) : col_free_index(cz0 * P + g, A.ncz, P, A.bcz);
        const bool pz = g >= 0 && lane_on && gz >= 0;
        const int zn = (gz < 0 ? 0 : gz) * plane_nodes;
#pragma unroll
        for (int j = 0; j < N; ++j) {
            const int yz = zn + (FAST ? YO(j) : max(YO(j), 0));
#pragma unroll
            for (int i = 0; i < N; ++i) {
                const int node = yz + (FAST ? XO(i) : max(XO(i), 0));
                if (FAST) u[j][i] = (ZISO || gz >= 0) ? __ldg(sp + (long long)node * A.rs) : (T)0;   // idle threads read plane 0 and drop it
                else u[j][i] = (pz && XO(i) >= 0 && YO(j) >= 0) ? __ldg(sp + (long long)node * A.rs) : (T)0;
            }
        }
    };

    // TMA: the owned nodes of cell t (src rows of both spins, this CTA's vectors) land in X buffer t % kColXBuf, their
    // nodal potential in its stage; nodes outside the mesh (Dirichlet faces) and vectors >= nvec are zero-filled. Issued
    // by one main thread as soon as phase B has consumed the buffer, so the expansion warps find their data waiting.
    auto issue_tma = [&](int t) {
        const int xb = t % kColXBuf;
        const unsigned xs = (unsigned)__cvta_generic_to_shared(xbase + xb * Cfg::XBYTES), vs = (unsigned)__cvta_generic_to_shared(vbase + xb * Cfg::VBYTES);
        const unsigned mbar = mbar0 + 8 * xb;
        const int bx0 = cx * P - (A.bcx == 0 ? 0 : 1), by0 = cy * P - (A.bcy == 0 ? 0 : 1), bz0 = (cz0 + t) * P - (A.bcz == 0 ? 0 : 1);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"((unsigned)(P * EPLANE * sizeof(T) + Cfg::VCELL * sizeof(double))) : "memory");
        asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                     ::"r"(xs), "l"(&A.tm_src), "r"(chunk * VPC * 2), "r"(bx0 * 2), "r"(by0), "r"(bz0), "r"(mbar) : "memory");
        asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                     ::"r"(vs), "l"(&A.tm_vb), "r"(bx0 * 4), "r"(by0), "r"(bz0), "r"(mbar) : "memory");
    };
    if constexpr (kMainTma)
        if (mtid == 0)
            for (int t = 0; t < kColXBuf && t < S; ++t) issue_tma(t);

    load_plane(plane_of(0));

    for (int t = 0; t < S; ++t) {
        // ------------------------------------------------------------------ phase A
        {
            const int g = plane_of(t);
            const bool act = g >= 0;
            const int slot = act ? g % N : 0;
            T* r1 = R1 + slot * PLANE + lane;
            T* r2 = R2 + slot * PLANE + lane;
            // with 32 lanes a warp is one plane: the warp whose plane is not new in this cell skips the phase
            if (!kWarpPlane || act) {
            // x-step bookkeeping: d[j] = uh . u[j][:]
            T d[N];
#pragma unroll
            for (int j = 0; j < N; ++j) {
                T s = (T)0;
#pragma unroll
                for (int i = 0; i < N; ++i) s = fma(UH(i), u[j][i], s);
                d[j] = s;
            }
            // output column i: a1 = (Ah u)[:, i], b1 = (Bx u)[:, i]; then the y-step on the column
#pragma unroll
            for (int i = 0; i < N; ++i) {
                const int ir = i;
                T a1[N], b1[N], b1s[N];
#pragma unroll
                for (int j = 0; j < N; ++j) {
                    T s = (T)0;
#pragma unroll
                    for (int ii = 0; ii < N; ++ii) s = fma(AH(i, ii), u[j][ii], s);
                    a1[j] = s;
                    b1[j] = fma(-UH(i), d[j], BETA(i) * u[j][i]);
                    b1s[j] = ZISO ? b1[j] : (T)A.rho_y * b1[j];
                }
                T da = (T)0, db = (T)0;
#pragma unroll
                for (int j = 0; j < N; ++j) { da = fma(UH(j), a1[j], da); db = fma(UH(j), b1[j], db); }
#pragma unroll
                for (int j = 0; j < N; ++j) {
                    T a2 = fma(-UH(j), da, BETA(j) * a1[j]);
#pragma unroll
                    for (int jj = 0; jj < N; ++jj) a2 = fma(AH(j, jj), b1s[jj], a2);
                    T b2 = fma(-UH(j), db, BETA(j) * b1[j]);
                    if (!ZISO) b2 *= (T)A.rho_z;
                    if (act) { r1[(j * N + ir) * L] = a2; r2[(j * N + ir) * L] = b2; }
                }
            }
            }
        }
        if (t + 1 < S) load_plane(plane_of(t + 1));          // in flight during phase B
        col_bar_sync(1, NTM);                                 // ring written
        col_bar_sync(2 + t % kColXBuf, Cfg::NTB);              // X(t) complete
        const T* X = reinterpret_cast<const T*>(xbase + (t % kColXBuf) * Cfg::XBYTES);
        // ------------------------------------------------------------------ phase B
        if (q_on) {
            const int j = q;
            const int cz = cz0 + t;
            const int s0 = (t * P) % N;                   // ring slot of local plane 0 of this cell
            int so[N], zn[N];
#pragma unroll
            for (int k = 0; k < N; ++k) {
                int sl = s0 + k; sl = sl >= N ? sl - N : sl;
                so[k] = sl;
                const int gz = col_free_index(cz * P + k, A.ncz, P, A.bcz);
                zn[k] = gz < 0 ? -1 : gz * plane_nodes;
            }
            const T* r1 = R1 + j * N * L + lane;
            const T* r2 = R2 + j * N * L + lane;
            const T* xp = X + j * P * L + lane;
#pragma unroll
            for (int i = 0; i < N; ++i) {
                const int ir = i;
                T f1[N], f2[N];
#pragma unroll
                for (int k = 0; k < N; ++k) {
                    f1[k] = r1[so[k] * PLANE + ir * L];
                    f2[k] = r2[so[k] * PLANE + ir * L];
                }
                T d1 = (T)0;
#pragma unroll
                for (int k = 0; k < N; ++k) d1 = fma(UH(k), f1[k], d1);
                T o[N];
#pragma unroll
                for (int k = 0; k < N; ++k) {
                    T s = fma(-UH(k), d1, BETA(k) * f1[k]);
#pragma unroll
                    for (int k2 = 0; k2 < N; ++k2) s = fma(AH(k, k2), f2[k2], s);
                    o[k] = s;
                }
                o[0] += carry[i];
                carry[i] = o[P];
                const bool xy_ok = FAST || (lane_on && XO(i) >= 0 && YO(j) >= 0);
                const int xy = FAST ? XO(i) + YO(j) : max(XO(i), 0) + max(YO(j), 0);
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    T v;
                    if (j < P && ir < P) v = fma(scax, o[k], (T)A.sc * xp[k * EPLANE + ir * L]);
                    else v = scax * o[k];
                    if (ZISO || (xy_ok && zn[k] >= 0)) col_red(dp + (long long)(xy + zn[k]) * A.rd, col_flip(v, sgn));
                }
                if (t == S - 1 && (ZISO || (xy_ok && zn[P] >= 0))) col_red(dp + (long long)(xy + zn[P]) * A.rd, col_flip((T)(scax * carry[i]), sgn));
            }
        }
        if constexpr (!kMainTma)
            if (t + kColXBuf < S) col_bar_arrive(4 + t % kColXBuf, Cfg::NTB);   // this X buffer is free
        col_bar_sync(1, NTM);                                 // ring and X(t) free
        if constexpr (kMainTma)
            if (mtid == 0 && t + kColXBuf < S) issue_tma(t + kColXBuf);
    }
#undef AH
#undef TAB_A
#undef TAB_U
#undef XO
#undef YO
#undef UH
#undef BETA
}

}  // namespace csf
