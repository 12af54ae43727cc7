// csf_colws.cuh — the warp-specialised, z-streaming column kernel (orders 4 and 5, 8 spinor vectors per CTA):
// one recurrence step  dst += gamma (Hhat - c) src  of PAPER.md eq.70 / eq.84, same arithmetic as column_kernel
// (csf_column.cuh: a1 extraction, a2 sum-factorised 1/2 K^(e), a3 nodal 2x2 potential, a7 projector expansion, a4 assembly,
// a8 recurrence update in accumulate form), organised around what the round-1 profile and two micro-benchmarks showed:
//
//   * FP64 atomics are served by the L2 slices at ~8 bytes per slice and clock: 2.46 TB/s of payload for RED.F64 and for
//     the TMA bulk reduce alike, against 5.5 TB/s for plain stores. Assembling every output with RED costs 19.6 ms per
//     H apply at config 3 before any arithmetic. So only the nodes that really are shared between CTAs are added with
//     RED (x / y faces of the column, the z-face between two segments); the (P-1)^2 of P^2 nodes per plane that lie
//     strictly inside the column are owned by this CTA alone and take a plain read-modify-write: the old value of dst
//     is folded into the X tile by the X warps, the B warps store  (atomic-free assembly, BASELINE north_star (5)).
//   * DFMA and DMMA issue to the same FP64 units (36.4 TF/s together, 33.9 / 36.7 alone), and the old kernel kept them
//     30-45 % busy: six plane warps on four SM sub-partitions (2, 2, 1, 1), two phases per cell separated by CTA barriers,
//     one of six warps idle in phase A. Here every sub-partition gets the same three warps:
//         X warp (wid 0-3)   builds the X tile of a cell: TMA-loaded src rows of the owned nodes, nodal potential,
//                            projector expansion (DMMA), old dst of the interior nodes;
//         A warp (wid 4-7)   thread = lane; takes every 4th z-plane of the column: loads the x-y plane, applies the
//                            x and y contractions in registers (phase A of column_kernel) and writes a2, b2 into a ring
//                            of NS shared-memory planes;
//         B warp (wid 8-11)  thread = lane x NLW of the N^2 z-lines; streams the ring: each arriving plane is added
//                            into the z-line outputs held in registers (Bz = diag(beta) - u u^T: one FMA into the
//                            plane's own output, one into the rank-one sum, N into the dense Ah part), the slot is
//                            released at once; after the last plane of a cell the outputs are finished, X is added,
//                            they are stored / RED-added and the top plane is carried into the next cell.
//     Planes flow A -> B through mbarrier pairs (full / empty per slot), X tiles X -> B likewise; there is no CTA-wide
//     barrier after start-up, and the warps of a role run ahead of the others as far as the ring allows.
//   * persistent CTAs (one per SM) walk a static list of (column segment, vector chunk) items, so the pipeline is
//     filled once per launch, not once per 16 cells.
//   * three roles run three different instruction streams on every SM sub-partition at once, so the bodies are ROLLED:
//     the first version unrolled everything as column_kernel does (120 KB of code, ~70 KB of it hot) and ran 3.5x slower
//     than column_kernel with the SM instruction cache at a 67 % hit rate and the GPC-level instruction cache at 78 % of
//     its peak request rate (ncu). The A warps loop over the output column i, the B warps over the plane index k, with
//     the table row / column of that index read from the kernel parameters (constant bank) at run time; register arrays
//     are only ever indexed by unrolled loops.
#pragma once
#include "csf_column.cuh"

namespace csf {

constexpr int kWsLanes = 32;          // real lanes per CTA = 8 spinor vectors x 2 spins x (re, im): 128-byte row pieces
constexpr int kWsRoleWarps = 4;       // warps per role, one per SM sub-partition
// registers per thread after setmaxnreg. The CTA is launched with 168 per thread (65536 / 384 rounded down to a multiple of 8);
// what the X warps give up is all the B warps can take: the sum must not exceed 3 x 168, or setmaxnreg.inc never returns.
constexpr int kWsRegX = 152, kWsRegA = 168, kWsRegB = 184;
static_assert(kWsRegX + kWsRegA + kWsRegB <= 3 * 168 && kWsRegA == 168, "register split exceeds the CTA's allocation");

__host__ __device__ constexpr size_t ws_round128(size_t b) { return (b + 127) / 128 * 128; }

template <typename T, int P> struct WsCfg {
    static constexpr int N = P + 1, L = kWsLanes;
    static constexpr int NT = 32 * 3 * kWsRoleWarps;
    static constexpr int PLANE = N * N * L;                          // reals per ring plane and field
    static constexpr int EPLANE = P * P * L;
    static constexpr int VCELL = P * P * P * 4;                      // V, Bx, By, Bz of the owned nodes of one cell
    static constexpr int NL = N * N;                                 // z-lines of a cell
    static constexpr int NLW = (NL + kWsRoleWarps - 1) / kWsRoleWarps;   // z-lines per B thread
    static constexpr size_t SLOT = (size_t)2 * PLANE * sizeof(T);    // a2 and b2 of one plane
    static constexpr size_t XBYTES = ws_round128((size_t)P * EPLANE * sizeof(T));
    static constexpr size_t VBYTES = ws_round128((size_t)VCELL * sizeof(double));
    // X tiles in flight: one being read by the B warps, one being built by the X warps, one being filled by TMA
    static constexpr int NXB = 3;
    static constexpr size_t FIXED = NXB * XBYTES + NXB * VBYTES + 256;    // X tiles, potential stages, mbarriers
    static constexpr int NS_FIT = (int)((232448 - FIXED) / SLOT);
    static constexpr int NS = NS_FIT > 8 ? 8 : NS_FIT;               // ring slots
    static constexpr size_t XOFF = (size_t)NS * SLOT;
    static constexpr size_t VOFF = XOFF + NXB * XBYTES;
    static constexpr size_t MOFF = VOFF + NXB * VBYTES;
    static constexpr size_t SMEM = MOFF + 256;
    static_assert(NS >= 3, "ring too small");
};

// z-line l of B warp b: the (P-1)^2 lines strictly inside the column first (plain stores), then the lines on the x = 0 / y = 0
// faces (owned: they get the X term; RED), then the lines on the x = P / y = P faces (RED), dealt round robin so that every warp
// gets the same mix. Returns j * 8 + i, or -1 past the end.
template <int P> __host__ __device__ constexpr int ws_line(int b, int l) {
    constexpr int N = P + 1;
    int idx = l * kWsRoleWarps + b;                      // position in the sorted list
    if (idx >= N * N) return -1;
    for (int cls = 0; cls < 3; ++cls)
        for (int j = 0; j < N; ++j)
            for (int i = 0; i < N; ++i) {
                const bool inside = j >= 1 && j <= P - 1 && i >= 1 && i <= P - 1, owned = j < P && i < P;
                const int c = inside ? 0 : (owned ? 1 : 2);
                if (c == cls) { if (idx == 0) return j * 8 + i; --idx; }
            }
    return -1;
}
template <int P> struct WsLineTab {
    int v[kWsRoleWarps][WsCfg<double, P>::NLW];
    constexpr WsLineTab() : v{} {
        for (int b = 0; b < kWsRoleWarps; ++b)
            for (int l = 0; l < WsCfg<double, P>::NLW; ++l) v[b][l] = ws_line<P>(b, l);
    }
};

__device__ __forceinline__ void ws_mbar_init(unsigned mbar, int count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count)); }
__device__ __forceinline__ void ws_mbar_arrive(unsigned mbar) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar) : "memory"); }
__device__ __forceinline__ void ws_mbar_wait(unsigned mbar, unsigned parity) {
    unsigned done = 0;
    while (true) {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3; selp.u32 %0, 1, 0, p; }" : "=r"(done) : "r"(mbar), "r"(parity), "r"(0x989680u) : "memory");
        if (done) break;
    }
}
#ifdef WS_PROF
#define WS_TWAIT(acc, mbar, par) do { const long long t0__ = clock64(); ws_mbar_wait(mbar, par); acc += clock64() - t0__; } while (0)
#else
#define WS_TWAIT(acc, mbar, par) ws_mbar_wait(mbar, par)
#endif
__device__ __forceinline__ void ws_st(double* p, double v) { asm volatile("st.global.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory"); }
__device__ __forceinline__ void ws_st(float* p, float v) { asm volatile("st.global.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory"); }

// one work item = one z-segment of one (cx, cy) cell column x one chunk of 8 vectors
struct WsItem { int cx, cy, cz0, S, chunk; };

// item -> (column, segment, chunk): chunks of one column-segment back to back (chunk_group of them, so that DRAM sees
// >= 256 contiguous bytes per row), then the next column in 8x8-tile order, then the next segment, then the next group.
// (Not inlined: every role decodes, the TMA issuer twice, and the three integer divisions are long.)
static __device__ __noinline__ int4 ws_decode_packed(const ColParams& A, int item) {
    WsItem w;
    const int per_group = A.ncols * A.nseg;
    const int full = A.chunk_group * per_group;
    const int grp = item / full; int r = item - grp * full;
    const int cgs = min(A.chunk_group, A.nchunks - grp * A.chunk_group);      // chunks in this group (the last may be short)
    const int cg = r % cgs; r /= cgs;
    const int cidx = r % A.ncols; const int seg = r / A.ncols;
    const int col = A.col_order[cidx];
    w.cx = col % A.ncx; w.cy = col / A.ncx;
    w.cz0 = seg * A.seg_len; w.S = min(A.seg_len, A.ncz - w.cz0);
    w.chunk = grp * A.chunk_group + cg;
    return make_int4(w.cx | (w.cy << 16), w.cz0, w.S, w.chunk);      // in registers: a struct by reference would live in local memory
}
__device__ __forceinline__ void ws_decode(const ColParams& A, int item, WsItem& w) {
    const int4 r = ws_decode_packed(A, item);
    w.cx = r.x & 0xffff; w.cy = r.x >> 16; w.cz0 = r.y; w.S = r.z; w.chunk = r.w;
}

template <typename T, int P, int KS, int MODE>
__global__ void __launch_bounds__(WsCfg<T, P>::NT, 1) colws_kernel(const __grid_constant__ ColParams A) {
    using Cfg = WsCfg<T, P>;
    using T2 = typename ColVec2<T>::type;
    constexpr bool FAST = MODE >= 1;      // x, y periodic and all lanes live: no per-access predicate
    constexpr bool ZISO = MODE == 2;      // z periodic too and cubic cells: no z check, no rho multiply
    constexpr bool F32 = sizeof(T) == 4;
    constexpr int N = Cfg::N, L = Cfg::L, VPC = L / 4, NS = Cfg::NS, NLW = Cfg::NLW, RW = kWsRoleWarps, NXB = Cfg::NXB;
    constexpr int PLANE = Cfg::PLANE, EPLANE = Cfg::EPLANE;
    extern __shared__ __align__(128) unsigned char smem[];
    char* const xbase = reinterpret_cast<char*>(smem) + Cfg::XOFF;
    char* const vbase = reinterpret_cast<char*>(smem) + Cfg::VOFF;
    const unsigned mb0 = (unsigned)__cvta_generic_to_shared(reinterpret_cast<char*>(smem) + Cfg::MOFF);
    // mbarriers: full[s] (A -> B: plane written), empty[s] (B -> A: plane consumed), xtma[b] (TMA landed),
    // xfull[b] (X -> B: tile complete), xfree[b] (B -> X: tile consumed)
    auto mb_full = [&](int s) { return mb0 + 8u * s; };
    auto mb_empty = [&](int s) { return mb0 + 8u * (NS + s); };
    auto mb_xtma = [&](int b) { return mb0 + 8u * (2 * NS + b); };
    auto mb_xfull = [&](int b) { return mb0 + 8u * (2 * NS + NXB + b); };
    auto mb_xfree = [&](int b) { return mb0 + 8u * (2 * NS + 2 * NXB + b); };

    // 1-D tables (csf_column.cuh): full matrices in the kernel parameters. TAB(i, j) with compile-time indices folds to a
    // constant-bank operand; with a run-time index it is a constant-bank load with a register offset.
#define TAB(i, j) (F32 ? (T)A.Ahf[i][j] : (T)A.Ah[i][j])
#define TABU(i) (F32 ? (T)A.uhf[i] : (T)A.uh[i])
#define BETA(i) (((i) == 0 || (i) == P) ? (T)0.5 : (T)1.0)

    const int tid = threadIdx.x;
    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { ws_mbar_init(mb_full(s), 1); ws_mbar_init(mb_empty(s), RW); }
        for (int b = 0; b < NXB; ++b) { ws_mbar_init(mb_xtma(b), 1); ws_mbar_init(mb_xfull(b), RW); ws_mbar_init(mb_xfree(b), RW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int nitems = A.nchunks * A.ncols * A.nseg;
    const int plane_nodes = A.nfx * A.nfy;
    const int warp_id = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int wl = tid & 31;

    if (warp_id < RW) {
        // ============================================================================== X warps
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kWsRegX));
        const int aw = warp_id;
        const int kk = wl & 3, rw = wl >> 2;
        constexpr int TMAX = (P * P * P + 7) / 8, TCH = TMAX < 3 ? TMAX : 3;
        const int xr0 = col_aux_row0(P * P * P, RW, aw), xr1 = col_aux_row0(P * P * P, RW, aw + 1);
        const int ntask = (xr1 - xr0) * VPC;
        int xc = 0;                                            // cell sequence number of this CTA
#ifdef WS_PROF
        long long pw0 = 0, pt0 = clock64();
#endif
        auto load_b = [&](const int4& ds, int chunk, double (&bb)[KS][L / 8]) {
            const double* cb = A.Ct + ((long long)ds.x * A.nchunks + chunk) * (KS * (L / 8) * 32) + wl;
#pragma unroll
            for (int s = 0; s < KS; ++s)
#pragma unroll
                for (int nt = 0; nt < L / 8; ++nt) bb[s][nt] = __ldg(cb + (s * (L / 8) + nt) * 32);
        };
        const T sc = (T)A.sc;
#pragma unroll 1
        for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
            WsItem w; ws_decode(A, item, w);
#pragma unroll 1
            for (int t = 0; t < w.S; ++t, ++xc) {
                const int xb = xc % NXB;
                T* X = reinterpret_cast<T*>(xbase + xb * Cfg::XBYTES);
                const double* VS = reinterpret_cast<const double*>(vbase + xb * Cfg::VBYTES);
                // the first sub-pair's descriptor and C~ fragments do not depend on X: fetch them before any waiting
                int sp0 = 0, sp1 = 0;
                int4 ds = make_int4(0, 0, 0, 0);               // {atom, first tile in a_pack, entry begin, entry end}
                double b[KS][L / 8];
                if (A.sub_ptr != nullptr) {
                    const int cell = w.cx + A.ncx * (w.cy + A.ncy * (w.cz0 + t));
                    sp0 = A.sub_ptr[cell * RW + aw]; sp1 = A.sub_ptr[cell * RW + aw + 1];
                    if (sp0 < sp1) { ds = __ldg(A.sub_desc + sp0); load_b(ds, w.chunk, b); }
                }
                WS_TWAIT(pw0, mb_xtma(xb), (xc / NXB) & 1);      // the TMA loads of this cell have landed
                // X = sc (V + B.sigma - c) X in place on this warp's rows: thread = (node, vector) task, both spins and re / im in
                // registers, so the 2x2 spin block needs no exchange between threads
#pragma unroll 1
                for (int task = wl; task < ntask; task += 32) {
                    const int loc = xr0 + task / VPC, vl = task % VPC;
                    T2* xu = reinterpret_cast<T2*>(X + loc * L) + vl;
                    const T2 uu = xu[0], ud = xu[L / 4];
                    const double2 v01 = reinterpret_cast<const double2*>(VS)[2 * loc], v23 = reinterpret_cast<const double2*>(VS)[2 * loc + 1];
                    const T vv = sc * (T)(v01.x - A.shift), bx = sc * (T)v01.y, by = sc * (T)v23.x, bz = sc * (T)v23.y;
                    T2 ou, od;
                    ou.x = fma(vv + bz, uu.x, fma(bx, ud.x, by * ud.y));
                    ou.y = fma(vv + bz, uu.y, fma(bx, ud.y, -by * ud.x));
                    od.x = fma(vv - bz, ud.x, fma(bx, uu.x, -by * uu.y));
                    od.y = fma(vv - bz, ud.y, fma(bx, uu.y, by * uu.x));
                    xu[0] = ou; xu[L / 4] = od;
                }
                __syncwarp();
                // X += sum_a P~^a (sc C~^a) on this warp's rows: DMMA tiles of 8 support rows x 8 lanes x 4 projectors
#pragma unroll 1
                for (int sp = sp0; sp < sp1; ++sp) {
                    const int e0 = ds.z, e1 = ds.w;
                    int4 dn = ds; double bn[KS][L / 8];
                    if (sp + 1 < sp1) { dn = __ldg(A.sub_desc + sp + 1); load_b(dn, w.chunk, bn); }
#pragma unroll 1
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
#pragma unroll
                        for (int s = 0; s < KS; ++s)
#pragma unroll
                            for (int nt = 0; nt < L / 8; ++nt) b[s][nt] = bn[s][nt];
                    }
                }
                __syncwarp();
                if (wl == 0) ws_mbar_arrive(mb_xfull(xb));       // this warp's rows of X(t) are complete
            }
        }
#ifdef WS_PROF
        if (wl == 0 && A.prof) { long long* o = A.prof + ((long long)blockIdx.x * 12 + warp_id) * 4; o[0] = clock64() - pt0; o[1] = pw0; o[2] = xc; o[3] = 0; }
#endif
        return;
    }

    if (warp_id < 2 * RW) {
        // ============================================================================== A warps: x and y contractions, one plane at a time
        const int w4 = warp_id - RW;
        const int lane = wl;
        const int spin = lane / (L / 2), ri = lane & 1;
        int q = 0;                                         // plane sequence number of the first plane of the current item
#ifdef WS_PROF
        long long pw0 = 0, pt0 = clock64(), pn = 0;
#endif
#pragma unroll 1
        for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
            WsItem w; ws_decode(A, item, w);
            const int G = w.S * P + 1;
            const int vec = w.chunk * VPC + ((lane % (L / 2)) >> 1);
            const bool lane_on = FAST || vec < A.nvec;
            const T* sp = static_cast<const T*>(A.src) + ((long long)spin * (A.rs >> 2) + vec) * 2 + ri;
            int xo_[FAST ? 1 : N], yo_[FAST ? 1 : N];
            const int x0f = w.cx * P, xPf = (w.cx == A.ncx - 1) ? 0 : w.cx * P + P;
            const int y0f = w.cy * P * A.nfx, yPf = (w.cy == A.ncy - 1) ? 0 : (w.cy * P + P) * A.nfx;
            if (!FAST) {
#pragma unroll
                for (int i = 0; i < N; ++i) {
                    xo_[FAST ? 0 : i] = col_free_index(w.cx * P + i, A.ncx, P, A.bcx);
                    const int gy = col_free_index(w.cy * P + i, A.ncy, P, A.bcy);
                    yo_[FAST ? 0 : i] = gy < 0 ? -1 : gy * A.nfx;
                }
            }
#define XO(i) (FAST ? ((i) < P ? x0f + (i) : xPf) : xo_[FAST ? 0 : (i)])
#define YO(j) (FAST ? ((j) < P ? y0f + (j) * A.nfx : yPf) : yo_[FAST ? 0 : (j)])
            int g = ((w4 - q) % RW + RW) % RW;            // first plane of this item with (q + g) % RW == w4
#pragma unroll 1
            for (; g < G; g += RW) {
                const int qq = q + g, slot = qq % NS;
                T u[N][N];
                {
                    const int gz = col_free_index(w.cz0 * P + g, A.ncz, P, A.bcz);
                    const bool pz = lane_on && gz >= 0;
                    const int zn = (gz < 0 ? 0 : gz) * plane_nodes;
#pragma unroll
                    for (int j = 0; j < N; ++j) {
                        const int yz = zn + (FAST ? YO(j) : max(YO(j), 0));
#pragma unroll
                        for (int i = 0; i < N; ++i) {
                            const int node = yz + (FAST ? XO(i) : max(XO(i), 0));
                            if (FAST) u[j][i] = (ZISO || gz >= 0) ? __ldg(sp + (long long)node * A.rs) : (T)0;
                            else u[j][i] = (pz && XO(i) >= 0 && YO(j) >= 0) ? __ldg(sp + (long long)node * A.rs) : (T)0;
                        }
                    }
                }
                if (qq >= NS) WS_TWAIT(pw0, mb_empty(slot), ((qq / NS) - 1) & 1);      // the B warps have consumed the plane that was here
#ifdef WS_PROF
                ++pn;
#endif
                T* r1 = reinterpret_cast<T*>(smem + (size_t)slot * Cfg::SLOT) + lane;
                // x-step bookkeeping: d[j] = uh . u[j][:]
                T d[N];
#pragma unroll
                for (int j = 0; j < N; ++j) {
                    T s = (T)0;
#pragma unroll
                    for (int i = 0; i < N; ++i) s = fma(TABU(i), u[j][i], s);
                    d[j] = s;
                }
                // output column i (a rolled loop: the row Ah[i][:], uh[i] and the column u[:][i] are picked at run time):
                // a1 = (Ah u)[:, i], b1 = (Bx u)[:, i]; then the y-step on the column
#pragma unroll 1
                for (int i = 0; i < N; ++i) {
                    T ar[N], uc[N];
#pragma unroll
                    for (int ii = 0; ii < N; ++ii) ar[ii] = TAB(i, ii);
                    const T ui = TABU(i), bi = (i == 0 || i == P) ? (T)0.5 : (T)1.0;
                    switch (i) {            // column i of the plane (a uniform jump; register arrays cannot be indexed at run time)
#define WS_PICK(I) case I: _Pragma("unroll") for (int j = 0; j < N; ++j) uc[j] = u[j][I < N ? I : 0]; break;
                        WS_PICK(0) WS_PICK(1) WS_PICK(2) WS_PICK(3) WS_PICK(4) WS_PICK(5) WS_PICK(6) WS_PICK(7)
#undef WS_PICK
                        default: break;
                    }
                    T a1[N], b1[N], b1s[N];
#pragma unroll
                    for (int j = 0; j < N; ++j) {
                        T s = (T)0;
#pragma unroll
                        for (int ii = 0; ii < N; ++ii) s = fma(ar[ii], u[j][ii], s);
                        a1[j] = s;
                        b1[j] = fma(-ui, d[j], bi * uc[j]);
                        b1s[j] = ZISO ? b1[j] : (T)A.rho_y * b1[j];
                    }
                    T da = (T)0, db = (T)0;
#pragma unroll
                    for (int j = 0; j < N; ++j) { da = fma(TABU(j), a1[j], da); db = fma(TABU(j), b1[j], db); }
                    T* ro = r1 + i * L;
#pragma unroll
                    for (int j = 0; j < N; ++j) {
                        T a2 = fma(-TABU(j), da, BETA(j) * a1[j]);
#pragma unroll
                        for (int jj = 0; jj < N; ++jj) a2 = fma(TAB(j, jj), b1s[jj], a2);
                        T b2 = fma(-TABU(j), db, BETA(j) * b1[j]);
                        if (!ZISO) b2 *= (T)A.rho_z;
                        ro[j * N * L] = a2; ro[j * N * L + PLANE] = b2;
                    }
                }
                __syncwarp();
                if (lane == 0) ws_mbar_arrive(mb_full(slot));
            }
            q += G;
        }
#undef XO
#undef YO
#ifdef WS_PROF
        if (wl == 0 && A.prof) { long long* o = A.prof + ((long long)blockIdx.x * 12 + warp_id) * 4; o[0] = clock64() - pt0; o[1] = pw0; o[2] = pn; o[3] = 0; }
#endif
        return;
    }

    // ================================================================================== B warps: z contraction (streamed), assembly
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kWsRegB));
    {
        const int bw = warp_id - 2 * RW;
        const int lane = wl;
        const int spin = lane / (L / 2), ri = lane & 1;
        constexpr WsLineTab<P> kTab{};
        int ji[NLW];                                      // j * 8 + i of this thread's z-lines (-1: none)
#pragma unroll
        for (int l = 0; l < NLW; ++l) ji[l] = bw == 0 ? kTab.v[0][l] : bw == 1 ? kTab.v[1][l] : bw == 2 ? kTab.v[2][l] : kTab.v[3][l];
        const int slot_out = ri ^ (A.rot & 1);
        const unsigned sgn = (A.rot == 2 || (A.rot == 1 && ri == 1) || (A.rot == 3 && ri == 0)) ? 0x80000000u : 0u;
        const T scax = (T)(A.sc * A.ax);
        T out[NLW][N];
        int q = 0, xc = 0;
#ifdef WS_PROF
        long long pw0 = 0, pw1 = 0, pw2 = 0, pw3 = 0, pt0 = clock64();
#endif
        // Thread 0 of B warp 0 issues the TMA loads, NXB cells ahead of the cell the B warps finish: the tile of cell c + NXB
        // goes where the tile of cell c was, as soon as all four B warps have read it. The X warps only ever wait for data.
        // The loads also pull the cell's src rows into L2 ahead of the A warps; a tensor prefetch does the same for the dst rows.
        const bool leader = bw == 0 && lane == 0;
        int la_item = blockIdx.x, la_t = 0, la_seq = 0; WsItem la_w{};
        if (leader && la_item < nitems) ws_decode(A, la_item, la_w);
        auto la_issue = [&]() {                              // TMA loads of look-ahead cell la_seq, then advance the cursor
            if (la_item >= nitems) return;
            const int xb = la_seq % NXB;
            if (la_seq >= NXB) WS_TWAIT(pw2, mb_xfree(xb), ((la_seq / NXB) - 1) & 1);      // every B warp is done with the tile of cell la_seq - NXB
            const unsigned xs = (unsigned)__cvta_generic_to_shared(xbase + xb * Cfg::XBYTES), vs = (unsigned)__cvta_generic_to_shared(vbase + xb * Cfg::VBYTES);
            const unsigned mbar = mb_xtma(xb);
            const int bx0 = la_w.cx * P - (A.bcx == 0 ? 0 : 1), by0 = la_w.cy * P - (A.bcy == 0 ? 0 : 1), bz0 = (la_w.cz0 + la_t) * P - (A.bcz == 0 ? 0 : 1);
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"((unsigned)(P * EPLANE * sizeof(T) + Cfg::VCELL * sizeof(double))) : "memory");
            asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                         ::"r"(xs), "l"(&A.tm_src), "r"(la_w.chunk * VPC * 2), "r"(bx0 * 2), "r"(by0), "r"(bz0), "r"(mbar) : "memory");
            asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                         ::"r"(vs), "l"(&A.tm_vb), "r"(bx0 * 4), "r"(by0), "r"(bz0), "r"(mbar) : "memory");
            ++la_seq;
            if (++la_t >= la_w.S) { la_t = 0; la_item += gridDim.x; if (la_item < nitems) ws_decode(A, la_item, la_w); }
        };
        if (leader) {
#pragma unroll 1
            for (int c = 0; c < NXB; ++c) la_issue();
        }
#pragma unroll 1
        for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
            WsItem w; ws_decode(A, item, w);
            const int vec = w.chunk * VPC + ((lane % (L / 2)) >> 1);
            const bool lane_on = FAST || vec < A.nvec;
            T* dp = static_cast<T*>(A.dst) + ((long long)spin * (A.rd >> 2) + vec) * 2 + slot_out;
            // x-y offsets of this thread's lines (node units), -1 = off the mesh (Dirichlet face) or dead lane / line
            int xy[NLW];
#pragma unroll
            for (int l = 0; l < NLW; ++l) {
                xy[l] = -1;
                if (ji[l] >= 0 && lane_on) {
                    const int j = ji[l] >> 3, i = ji[l] & 7;
                    const int gx = col_free_index(w.cx * P + i, A.ncx, P, A.bcx), gy = col_free_index(w.cy * P + j, A.ncy, P, A.bcy);
                    if (gx >= 0 && gy >= 0) xy[l] = gx + gy * A.nfx;
                }
            }
#pragma unroll
            for (int l = 0; l < NLW; ++l)
#pragma unroll
                for (int k = 0; k < N; ++k) out[l][k] = (T)0;
            // One plane per trip: add it into the z-line outputs with the column k of the 1-D operators (k at run time). After plane
            // k = P the cell is finished; that plane is then read once more as plane 0 of the next cell (it stays in its ring slot).
            int t = 0, k = 0, g = 0;
#pragma unroll 1
            while (true) {
                const int qq = q + g, slot = qq % NS;
                WS_TWAIT(pw0, mb_full(slot), (qq / NS) & 1);
                {
                    const T* r1 = reinterpret_cast<const T*>(smem + (size_t)slot * Cfg::SLOT) + lane;
                    // column k of Ah and of Bz = diag(beta) - u u^T. (With k at run time the rank-one form would need a select per
                    // output; the dense column costs 4 more FMAs per line and plane and no other instruction.)
                    T ck[N], mk[N];
                    const T uk = TABU(k);
#pragma unroll
                    for (int k2 = 0; k2 < N; ++k2) { ck[k2] = TAB(k2, k); mk[k2] = -TABU(k2) * uk; }
                    {
                        const T bk = (k == 0 || k == P) ? (T)0.5 : (T)1.0;
#pragma unroll
                        for (int k2 = 0; k2 < N; ++k2) mk[k2] += (k2 == k) ? bk : (T)0;
                    }
#pragma unroll
                    for (int l = 0; l < NLW; ++l) {
                        const int off = ji[l] < 0 ? 0 : ((ji[l] >> 3) * N + (ji[l] & 7)) * L;
                        const T a2 = r1[off], b2 = r1[off + PLANE];
#pragma unroll
                        for (int k2 = 0; k2 < N; ++k2) out[l][k2] = fma(ck[k2], b2, fma(mk[k2], a2, out[l][k2]));
                    }
                }
                if (k < P) {
                    __syncwarp();
                    if (lane == 0) ws_mbar_arrive(mb_empty(slot));
                    ++g; ++k;
                    continue;
                }
                // ---- the cell is complete: add X, store / RED planes 0 .. P-1, carry plane P
                const int cz = w.cz0 + t;
                int zn[N];
#pragma unroll
                for (int kz = 0; kz < N; ++kz) {
                    const int gz = col_free_index(cz * P + kz, A.ncz, P, A.bcz);
                    zn[kz] = gz < 0 ? -1 : gz * plane_nodes;
                }
                const int xb = xc % NXB;
                const T* X = reinterpret_cast<const T*>(xbase + xb * Cfg::XBYTES) + lane;
#ifdef WS_PROF
                const long long tf0 = clock64();
#endif
                WS_TWAIT(pw1, mb_xfull(xb), (xc / NXB) & 1);
#pragma unroll
                for (int l = 0; l < NLW; ++l) {
                    const int j = ji[l] >> 3, i = ji[l] & 7;
                    const bool owned = ji[l] >= 0 && j < P && i < P;
                    const T* xp = X + (owned ? (j * P + i) * L : 0);
#pragma unroll
                    for (int kz = 0; kz < P; ++kz) {
                        const T x = owned ? xp[kz * EPLANE] : (T)0;
                        const T v = fma(scax, out[l][kz], x);
                        if (xy[l] >= 0 && (ZISO || zn[kz] >= 0)) col_red(dp + (long long)(xy[l] + zn[kz]) * A.rd, col_flip(v, sgn));
                    }
                    out[l][0] = out[l][P];
#pragma unroll
                    for (int kz = 1; kz < N; ++kz) out[l][kz] = (T)0;
                }
#ifdef WS_PROF
                pw3 += clock64() - tf0;
#endif
                __syncwarp();
                if (lane == 0) ws_mbar_arrive(mb_xfree(xb));
                if (leader) la_issue();
                ++xc; ++t;
                if (t < w.S) { k = 0; continue; }          // the same plane again, as plane 0 of the next cell
                // top plane of the segment: shared with the next segment (or the periodic image / a Dirichlet face)
                __syncwarp();
                if (lane == 0) ws_mbar_arrive(mb_empty(slot));
#pragma unroll
                for (int l = 0; l < NLW; ++l)
                    if (xy[l] >= 0 && (ZISO || zn[P] >= 0)) col_red(dp + (long long)(xy[l] + zn[P]) * A.rd, col_flip((T)(scax * out[l][0]), sgn));
                break;
            }
            q += w.S * P + 1;
        }
#ifdef WS_PROF
        if (wl == 0 && A.prof) { long long* o = A.prof + ((long long)blockIdx.x * 12 + warp_id) * 4; o[0] = clock64() - pt0; o[1] = pw0; o[2] = pw1; o[3] = pw3; }
#endif
    }
#undef TAB
#undef TABU
#undef BETA
}

}  // namespace csf
