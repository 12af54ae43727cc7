// csf_kernels.cuh — hand-written sm_100a kernels of the Chebyshev-filtered spinor H.X.
//
// One recurrence step is  dst += gamma (Hhat - c) src  with gamma = sc * i^rot  ("accumulate form":
// with W_k = i^(m-k) T_k(H~) X the three-term recurrence of PAPER.md eq.70 becomes
// W_{k+1} = W_{k-1} + (-2i/e)(Hhat - c) W_k, a pure accumulation into the buffer that holds W_{k-1};
// multiplying by a power of i is exact in binary floating point). Per step three kernels run:
//
//   proj_gather_kernel   C^a  = P~^aT src|supp(a)                     (eq.84 inner sum, a5)
//   delta_apply_kernel   C~^a = Delta^{gamma_a} C^a                   (eq.76, a6)
//   cell_kernel          gather -> sum-factorised 1/2 K -> nodal 2x2 potential, shift and projector
//                        expansion on the nodes the cell owns -> scaled scatter-add   (a1-a4, a7, a8)
//
// Data layout: multivector element (node I, spin s, vector v) = complex128 at [(2I+s)*ld + v]. The operator
// tables are real, so the real and imaginary parts are independent batch entries: a "lane" is one double of
// the (spin, vector, re/im) batch, lanes of a warp cover contiguous 8-byte words of one or two 128-byte
// segments (fully coalesced), and the spin 2x2 potential is applied with warp shuffles between lanes.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace csf {

constexpr int kTabN = 8;

struct CellParams {
    // Loewdin-scaled 1-D operators (csf_tables.h). Ax, bxs, uxs carry the step scale sc.
    double Ay[kTabN][kTabN], Az[kTabN][kTabN], Ax[kTabN][kTabN];
    double by[kTabN], uy[kTabN], bz[kTabN], uz[kTabN], bxs[kTabN], ux[kTabN], uxs[kTabN];
    const double* src; double* dst;
    long long ld_src, ld_dst; int nvec;
    int ncx, ncy, ncz, nfx, nfy, nfz, bcx, bcy, bcz;
    const int* cell_order; int ncells;
    const double* vb;        // [M][4] = V, Bx, By, Bz at the nodes
    double shift;            // c of (Hhat - c)
    double sc; int rot;      // gamma = sc * i^rot
    // projector expansion (cell-major view of the entry list)
    const int* pair_ptr;     // [ncells+1]
    const int* pair_atom;    // [npairs]
    const int* pair_off;     // [npairs][P+1] entry ranges per owned z-plane
    const int* ent_loc;      // [nent] local index j*P+i inside the owned plane
    const double* ent_p;     // [nent][npjp] S_I P_{I chi}
    const long long* atom_coff;  // [natoms] row offset of atom a in C / C~ (rows 2 chi + s)
    const int* atom_npj;     // [natoms]
    const double* Ct;        // C~ [rows][ldc] complex128
    long long ldc; int npjp;
};

__device__ __forceinline__ double flip_sign(double x, unsigned mask) {
    return __hiloint2double(__double2hiint(x) ^ (int)mask, __double2loint(x));
}

// free (unconstrained) 1-D node index of full index f, or -1 on a Dirichlet face
__device__ __forceinline__ int free_index(int f, int ncell, int p, int bc) {
    const int nfull = ncell * p;
    if (bc == 0) return f >= nfull ? f - nfull : f;
    return (f == 0 || f == nfull) ? -1 : f - 1;
}

// ---------------------------------------------------------------------------------------------------
// cell kernel: one CTA = one cell x (L/4) vectors x 2 spins. Thread (plane, lane).
//   phase 1: plane = z index; the thread holds the x-y plane X[j][i] of its lane in registers,
//            F1 = By X (rank-one form), F2 = Ay X (dense) -> shared memory;
//            on owned nodes E = (V + B.sigma - c) x + sum_a P~ C~^a  -> shared memory.
//   phase 2: plane = y index; per x-column the z-operators, then the x-operators row by row:
//            out = Ax (Bz F1) + Bx (Bz F2 + Az F1) + sc E, scatter-added with RED.F64.
// ---------------------------------------------------------------------------------------------------
template <int P, int L, int NPJ>
__global__ void __launch_bounds__((P + 1) * L) cell_kernel(const __grid_constant__ CellParams A) {
    constexpr int N = P + 1;
    extern __shared__ double smem[];
    double* F1 = smem;
    double* F2 = smem + N * N * N * L;
    double* E = smem + 2 * N * N * N * L;

    const int tid = threadIdx.x;
    const int lane = tid % L;
    const int plane = tid / L;
    const unsigned wmask = __activemask();

    const int nchunk_v = L / 4;
    const int cidx = blockIdx.x % A.ncells;
    const int chunk = blockIdx.x / A.ncells;
    const int cell = A.cell_order[cidx];
    const int cx = cell % A.ncx, cy = (cell / A.ncx) % A.ncy, cz = cell / (A.ncx * A.ncy);

    const int spin = lane / (L / 2);
    const int ri = lane & 1;
    const int vec = chunk * nchunk_v + ((lane % (L / 2)) >> 1);
    const bool lane_on = vec < A.nvec;

    int gx[N], gy[N], gz[N];
#pragma unroll
    for (int i = 0; i < N; ++i) {
        gx[i] = free_index(cx * P + i, A.ncx, P, A.bcx);
        gy[i] = free_index(cy * P + i, A.ncy, P, A.bcy);
        gz[i] = free_index(cz * P + i, A.ncz, P, A.bcz);
    }
    const long long rs = 4 * A.ld_src;                               // doubles per node (2 rows)
    const long long lane_off = ((long long)spin * A.ld_src + vec) * 2 + ri;

    // ------------------------------------------------------------------ phase 1
    {
        const int k = plane;
        double x[N][N];
        const double* sp = A.src + lane_off;
#pragma unroll
        for (int j = 0; j < N; ++j)
#pragma unroll
            for (int i = 0; i < N; ++i) {
                const bool ok = lane_on && gx[i] >= 0 && gy[j] >= 0 && gz[k] >= 0;
                const int node = gx[i] + A.nfx * (gy[j] + A.nfy * gz[k]);
                x[j][i] = ok ? __ldg(sp + (long long)node * rs) : 0.0;
            }
        // y-operators, column by column
#pragma unroll
        for (int i = 0; i < N; ++i) {
            double d = 0.0;
#pragma unroll
            for (int j = 0; j < N; ++j) d = fma(A.uy[j], x[j][i], d);
#pragma unroll
            for (int j = 0; j < N; ++j) {
                double f1 = fma(-A.uy[j], d, A.by[j] * x[j][i]);
                double f2 = 0.0;
#pragma unroll
                for (int jj = 0; jj < N; ++jj) f2 = fma(A.Ay[j][jj], x[jj][i], f2);
                F1[((k * N + j) * N + i) * L + lane] = f1;
                F2[((k * N + j) * N + i) * L + lane] = f2;
            }
        }
        // nodal terms on the nodes this cell owns (local index < P in every direction)
        const double sz = spin ? -1.0 : 1.0;
        const double sy = (spin == ri) ? 1.0 : -1.0;
#pragma unroll
        for (int j = 0; j < P; ++j)
#pragma unroll
            for (int i = 0; i < P; ++i) {
                const double own = x[j][i];
                const double t1 = __shfl_xor_sync(wmask, own, L / 2);   // other spin, same re/im
                const double t2 = __shfl_xor_sync(wmask, t1, 1);        // other spin, other re/im
                if (k < P) {
                    double e = 0.0;
                    if (gx[i] >= 0 && gy[j] >= 0 && gz[k] >= 0) {
                        const int node = gx[i] + A.nfx * (gy[j] + A.nfy * gz[k]);
                        const double2 v01 = __ldg(reinterpret_cast<const double2*>(A.vb) + 2 * (long long)node);
                        const double2 v23 = __ldg(reinterpret_cast<const double2*>(A.vb) + 2 * (long long)node + 1);
                        e = fma(v01.x - A.shift + sz * v23.y, own, fma(v01.y, t1, sy * v23.x * t2));
                    }
                    E[((k * P + j) * P + i) * L + lane] = e;
                }
            }
        // projector expansion  E += sum_a P~^a C~^a  on owned nodes of this z-plane
        if (k < P && A.pair_ptr != nullptr) {
            const int pr0 = A.pair_ptr[cell], pr1 = A.pair_ptr[cell + 1];
            for (int pr = pr0; pr < pr1; ++pr) {
                const int e0 = A.pair_off[pr * (P + 1) + k], e1 = A.pair_off[pr * (P + 1) + k + 1];
                if (e0 == e1) continue;
                const int atom = A.pair_atom[pr];
                const double* cb = A.Ct + ((A.atom_coff[atom] + spin) * A.ldc + vec) * 2 + ri;
                if (NPJ > 0) {
                    double ct[NPJ > 0 ? NPJ : 1];
#pragma unroll
                    for (int c = 0; c < NPJ; ++c) ct[c] = lane_on ? __ldg(cb + (long long)c * 4 * A.ldc) : 0.0;
                    for (int e = e0; e < e1; ++e) {
                        const double2* pp = reinterpret_cast<const double2*>(A.ent_p + (long long)e * A.npjp);
                        double acc = 0.0;
#pragma unroll
                        for (int c = 0; c < NPJ / 2; ++c) { const double2 pv = __ldg(pp + c); acc = fma(pv.x, ct[2 * c], acc); acc = fma(pv.y, ct[2 * c + 1], acc); }
                        E[(k * P * P + A.ent_loc[e]) * L + lane] += acc;
                    }
                } else {
                    const int npj = A.atom_npj[atom];
                    for (int e = e0; e < e1; ++e) {
                        const double* pp = A.ent_p + (long long)e * A.npjp;
                        double acc = 0.0;
                        for (int c = 0; c < npj; ++c) acc = fma(__ldg(pp + c), lane_on ? __ldg(cb + (long long)c * 4 * A.ldc) : 0.0, acc);
                        E[(k * P * P + A.ent_loc[e]) * L + lane] += acc;
                    }
                }
            }
        }
    }
    __syncthreads();
    // ------------------------------------------------------------------ phase 2
    {
        const int j = plane;
        double a[N][N], g[N][N];     // [k][i]
#pragma unroll
        for (int i = 0; i < N; ++i) {
            double f1[N], f2[N];
#pragma unroll
            for (int k = 0; k < N; ++k) { f1[k] = F1[((k * N + j) * N + i) * L + lane]; f2[k] = F2[((k * N + j) * N + i) * L + lane]; }
            double d1 = 0.0, d2 = 0.0;
#pragma unroll
            for (int k = 0; k < N; ++k) { d1 = fma(A.uz[k], f1[k], d1); d2 = fma(A.uz[k], f2[k], d2); }
#pragma unroll
            for (int k = 0; k < N; ++k) {
                a[k][i] = fma(-A.uz[k], d1, A.bz[k] * f1[k]);
                double t = fma(-A.uz[k], d2, A.bz[k] * f2[k]);
#pragma unroll
                for (int kk = 0; kk < N; ++kk) t = fma(A.Az[k][kk], f1[kk], t);
                g[k][i] = t;
            }
        }
        // multiplication by i^rot: swap re/im slot and flip signs (exact)
        const int slot = ri ^ (A.rot & 1);
        const unsigned sgn = (A.rot == 2 || (A.rot == 1 && ri == 1) || (A.rot == 3 && ri == 0)) ? 0x80000000u : 0u;
        double* dp = A.dst + ((long long)spin * A.ld_dst + vec) * 2 + slot;
        const long long rd = 4 * A.ld_dst;
#pragma unroll
        for (int k = 0; k < N; ++k) {
            double dg = 0.0;
#pragma unroll
            for (int i = 0; i < N; ++i) dg = fma(A.ux[i], g[k][i], dg);
#pragma unroll
            for (int i = 0; i < N; ++i) {
                double o = fma(-A.uxs[i], dg, A.bxs[i] * g[k][i]);
#pragma unroll
                for (int ii = 0; ii < N; ++ii) o = fma(A.Ax[i][ii], a[k][ii], o);
                if (k < P && j < P && i < P) o = fma(A.sc, E[((k * P + j) * P + i) * L + lane], o);
                if (lane_on && gx[i] >= 0 && gy[j] >= 0 && gz[k] >= 0) {
                    const int node = gx[i] + A.nfx * (gy[j] + A.nfy * gz[k]);
                    atomicAdd(dp + (long long)node * rd, flip_sign(o, sgn));
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// proj_gather_kernel: C[atom][2 chi + s][v] += sum_{I in block's node range} P~_{I chi} src[(2I+s)][v].
// grid.x = gather blocks (atom, node range), grid.y = vector chunks of 8; 4 warps split the nodes,
// shared-memory reduce, one RED per (chi, lane).
// ---------------------------------------------------------------------------------------------------
struct GatherParams {
    const double* src; long long ld; int nvec;
    const int* gb_atom; const int* gb_beg; const int* gb_end;   // gather blocks over the entry list
    const int* ent_node; const double* ent_p; int npjp;
    const long long* atom_coff; const int* atom_npj;
    double* C; long long ldc;
};

template <int NPJ>
__global__ void __launch_bounds__(128) proj_gather_kernel(const __grid_constant__ GatherParams A) {
    constexpr int NA = NPJ > 0 ? NPJ : 32;
    __shared__ double red[3][NA][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int spin = lane >> 4, ri = lane & 1;
    const int vec = blockIdx.y * 8 + ((lane & 15) >> 1);
    const bool lane_on = vec < A.nvec;
    const int atom = A.gb_atom[blockIdx.x];
    const int e0 = A.gb_beg[blockIdx.x], e1 = A.gb_end[blockIdx.x];
    const int npj = NPJ > 0 ? NPJ : A.atom_npj[atom];
    const double* sp = A.src + ((long long)spin * A.ld + vec) * 2 + ri;
    const long long rs = 4 * A.ld;
    double acc[NA];
#pragma unroll
    for (int c = 0; c < NA; ++c) acc[c] = 0.0;
    for (int e = e0 + warp; e < e1; e += 4) {
        const double xv = lane_on ? __ldg(sp + (long long)A.ent_node[e] * rs) : 0.0;
        if (NPJ > 0) {
            const double2* pp = reinterpret_cast<const double2*>(A.ent_p + (long long)e * A.npjp);
#pragma unroll
            for (int c = 0; c < NPJ / 2; ++c) { const double2 pv = __ldg(pp + c); acc[2 * c] = fma(pv.x, xv, acc[2 * c]); acc[2 * c + 1] = fma(pv.y, xv, acc[2 * c + 1]); }
        } else {
            const double* pp = A.ent_p + (long long)e * A.npjp;
#pragma unroll
            for (int c = 0; c < NA; ++c) if (c < npj) acc[c] = fma(__ldg(pp + c), xv, acc[c]);
        }
    }
    if (warp > 0) {
#pragma unroll
        for (int c = 0; c < NA; ++c) red[warp - 1][c][lane] = acc[c];
    }
    __syncthreads();
    if (warp == 0 && lane_on) {
        double* cp = A.C + ((A.atom_coff[atom] + spin) * A.ldc + vec) * 2 + ri;
#pragma unroll
        for (int c = 0; c < NA; ++c) {
            if (c < npj) {
                const double s = acc[c] + red[0][c][lane] + red[1][c][lane] + red[2][c][lane];
                atomicAdd(cp + (long long)c * 4 * A.ldc, s);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// delta_apply_kernel: Ct[a][r][v] = sum_q Delta_t[r][q] C[a][q][v], r, q = 2 chi + s  (eq.76)
// grid = (atoms, vector chunks of 32); thread = (row group, vector).
// ---------------------------------------------------------------------------------------------------
struct DeltaParams {
    const double2* C; double2* Ct; long long ldc; int nvec;
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
        A.Ct[(base + r) * A.ldc + v] = make_double2(sr, si);
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

}  // namespace csf
