// csf_dense.cuh — the general-quadrature potential and the dense cell-matrix form of H X.
//
//   PAPER.md:528-547 eq.79-83: with the potential given at the n_q^3 Gauss-Legendre points of every cell, the cell-level
//   potential matrices are V^(e) = (N~ o (w J v^(e))) N~^T, dense n_p^3 x n_p^3, N~[a][q] = N~_a(r~_q).
//   PAPER.md:551-561 eq.84: H X cell by cell: extract X^(e) = R^(e) X, multiply by the dense cell-level matrix,
//   assemble Y += R^(e)T Y^(e), add the nonlocal part C^T Delta C X.
//
// This is the paper's own formulation of the local part (one dense 2 n_p^3 x 2 n_p^3 block per cell, batched GEMM),
// built here as the measured alternative to the sum-factorised column kernel of csf_column.cuh, and as the only path
// that takes a non-nodal quadrature rule. Every cell matrix carries the Loewdin scaling S^(e) (.) S^(e) and the kinetic
// block 1/2 K^(e) (the same for all cells of the uniform mesh):
//      H^(e) = [ P   M1 - i M2 ]     P  = 1/2 K + V + Bz,   Q  = 1/2 K + V - Bz,
//              [ M1 + i M2   Q ]     M1 = Bx,               M2 = By          (sigma of P:46; all four real, symmetric)
// The four real matrices of a cell are stored in the order the FP64 tensor-core tile (mma.sync m8n8k4) reads its
// A operand:  [cell][m-tile of 8 rows][k-step of 4 columns][matrix P, Q, M1, M2][lane = (row % 8) * 4 + column % 4],
// so that a warp fetches the four fragments of one (m-tile, k-step) as 1 KB of consecutive memory.
#pragma once
#include <cuda_runtime.h>

namespace csf {

// ---------------------------------------------------------------------------------------------------------------------
// set-up: the cell matrices from the potential at the quadrature points
struct CellMatParams {
    const double* Ns;        // [nq3][n3p]: s_a N~_a(r~_q), s_a = (1-D lumped masses of node a)^(-1/2); zero for a >= n3
    const double* wJ;        // [nq3]: w_q J^(e)
    const double* kin;       // [n3p][n3p]: S^(e) 1/2 K^(e) S^(e)
    const double* vq;        // [E][nq3][4]: V_eff, B_x, B_y, B_z at the quadrature points
    double* out;             // fragment order, see above
    int nq3, n3, n3p;
    double vshift;           // added to V_eff at every quadrature point (|k|^2/2 of the k-point Hamiltonian)
};

constexpr int kCmChunk = 128;     // quadrature points staged per pass

// grid = cells x m-tiles (m-tile fastest), 256 threads: thread = column b (strided), 8 rows x 4 fields in registers
__global__ void __launch_bounds__(256) cellmat_build_kernel(const __grid_constant__ CellMatParams A) {
    __shared__ double f[kCmChunk][4];
    __shared__ double na[kCmChunk][8];
    const int mtn = A.n3p / 8, ksn = A.n3p / 4;
    const int mt = blockIdx.x % mtn; const long long e = blockIdx.x / mtn;
    for (int b0 = 0; b0 < A.n3p; b0 += 256) {
        const int b = b0 + threadIdx.x;
        double acc[8][4];
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int d = 0; d < 4; ++d) acc[r][d] = 0.0;
        for (int q0 = 0; q0 < A.nq3; q0 += kCmChunk) {
            const int nqc = min(kCmChunk, A.nq3 - q0);
            __syncthreads();
            for (int t = threadIdx.x; t < nqc * 4; t += 256) f[t >> 2][t & 3] = A.wJ[q0 + (t >> 2)] * (A.vq[(e * A.nq3 + q0 + (t >> 2)) * 4 + (t & 3)] + ((t & 3) == 0 ? A.vshift : 0.0));
            for (int t = threadIdx.x; t < nqc * 8; t += 256) na[t >> 3][t & 7] = A.Ns[(long long)(q0 + (t >> 3)) * A.n3p + mt * 8 + (t & 7)];
            __syncthreads();
            if (b < A.n3p)
                for (int q = 0; q < nqc; ++q) {
                    const double nb = A.Ns[(long long)(q0 + q) * A.n3p + b];
                    const double g0 = nb * f[q][0], g1 = nb * f[q][1], g2 = nb * f[q][2], g3 = nb * f[q][3];
#pragma unroll
                    for (int r = 0; r < 8; ++r) {
                        const double a = na[q][r];
                        acc[r][0] = fma(a, g0, acc[r][0]); acc[r][1] = fma(a, g1, acc[r][1]);
                        acc[r][2] = fma(a, g2, acc[r][2]); acc[r][3] = fma(a, g3, acc[r][3]);
                    }
                }
        }
        if (b < A.n3p) {
            double* o = A.out + (((e * mtn + mt) * ksn + (b >> 2)) * 4) * 32 + (b & 3);
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const double k = A.kin[(long long)(mt * 8 + r) * A.n3p + b];
                o[0 * 32 + r * 4] = k + acc[r][0] + acc[r][3];
                o[1 * 32 + r * 4] = k + acc[r][0] - acc[r][3];
                o[2 * 32 + r * 4] = acc[r][1];
                o[3 * 32 + r * 4] = acc[r][2];
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// eq.84: extraction, dense cell-level product, assembly
struct DenseParams {
    const double* mat;                 // cell matrices in fragment order
    const double2* X; long long ld;    // [2M][ld] complex128
    double* Y; long long ldy;          // [2M][ldy] complex128 as reals; Y += ...
    int nvec, p, n3, n3p;
    int ncx, ncy, ncz, nfx, nfy, nfz, bcx, bcy, bcz;      // bc: 0 periodic, 1 Dirichlet (boundary nodes removed)
    double fr, fi;                     // Y += f (H^(e) X^(e)), f = fr + i fi (1 for a plain apply; sc i^rot for a recurrence step)
    const double* gk;                  // KPT: S^(e) sum_d k_d G_d^(e) S^(e), G_d[a][b] = int N_a d_d N_b, fragment order [m-tile][k-step][32]; the same for all cells
};

__device__ __forceinline__ void dense_dmma(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// global index of the 1-D node f = cell * p + i of a direction with nc cells, or -1 on a Dirichlet face
__device__ __forceinline__ int dense_axis_node(int f, int nc, int p, int bc) {
    if (bc == 0) return f == nc * p ? 0 : f;
    return (f == 0 || f == nc * p) ? -1 : f - 1;
}

// VC spinor vectors per CTA; the X tile of the cell is kept as two real arrays [n3p][LDW] (spin up, spin down). The B fragment
// of a DMMA is read as (row k0 + lane % 4, column n0 + lane / 4): a half-warp must land in 16 different 8-byte banks, i.e.
// the four rows must start 4 doubles apart mod 16. VC = 8: row stride 2 VC + 4 = 20. VC = 16: stride 32 with the column
// XOR-ed by 4 (row % 4) instead of padding, so that the tile of an order-5 cell (110 KB) leaves room for two CTAs per SM.
template <int VC> __host__ __device__ constexpr int dense_ldw() { return VC == 16 ? 32 : 2 * VC + 4; }
template <int VC> __host__ __device__ constexpr int dense_col(int row, int col) { return VC == 16 ? (col ^ ((row & 3) * 4)) : col; }
template <int VC> __host__ __device__ constexpr size_t dense_smem(int n3p) { return (size_t)2 * n3p * dense_ldw<VC>() * sizeof(double) + (size_t)n3p * sizeof(int); }

// grid = cells x vector chunks (chunk fastest): the chunks of one cell run next to each other, so the cell's matrices (1.5 MB at order 5)
// are fetched from HBM once and served from L2 to the other chunks. 8 warps, warp w takes the m-tiles w, w + 8, ...
// KPT: the Bloch term -i k.grad of eq.40, spin-diagonal: Yu -= i Gk Xu, Yd -= i Gk Xd; it joins the two accumulators
// that are multiplied by -+ i anyway: T2 = M2 Xd + Gk Xu, T1 = M2 Xu - Gk Xd.
template <int VC, bool KPT>
__global__ void __launch_bounds__(256, 2) dense_cell_kernel(const __grid_constant__ DenseParams A) {
    constexpr int LDW = dense_ldw<VC>(), NT = VC / 4;          // n-tiles of 8 real columns = 4 complex vectors
    extern __shared__ __align__(16) unsigned char dense_raw[];
    double* Xu = reinterpret_cast<double*>(dense_raw);
    double* Xd = Xu + (size_t)A.n3p * LDW;
    int* node = reinterpret_cast<int*>(Xd + (size_t)A.n3p * LDW);
    const int nch = (A.nvec + VC - 1) / VC;
    const int e = blockIdx.x / nch, v0 = (blockIdx.x % nch) * VC;
    const int n = A.p + 1;
    const int cx = e % A.ncx, cy = (e / A.ncx) % A.ncy, cz = e / (A.ncx * A.ncy);
    // connectivity of the cell (eq.74), local node a = i + n (j + n k)
    for (int a = threadIdx.x; a < A.n3p; a += 256) {
        int g = -1;
        if (a < A.n3) {
            const int i = a % n, j = (a / n) % n, k = a / (n * n);
            const int gx = dense_axis_node(cx * A.p + i, A.ncx, A.p, A.bcx), gy = dense_axis_node(cy * A.p + j, A.ncy, A.p, A.bcy),
                      gz = dense_axis_node(cz * A.p + k, A.ncz, A.p, A.bcz);
            if (gx >= 0 && gy >= 0 && gz >= 0) g = gx + A.nfx * (gy + A.nfy * gz);
        }
        node[a] = g;
    }
    __syncthreads();
    // step 1, extraction: X^(e) = R^(e) X
    for (int t = threadIdx.x; t < A.n3p * 2 * VC; t += 256) {
        const int c = t % VC, s = (t / VC) & 1, a = t / (2 * VC);
        const int g = node[a];
        double2 z = make_double2(0.0, 0.0);
        if (g >= 0 && v0 + c < A.nvec) z = A.X[(2LL * g + s) * A.ld + v0 + c];
        *reinterpret_cast<double2*>((s ? Xd : Xu) + (size_t)a * LDW + dense_col<VC>(a, 2 * c)) = z;
    }
    __syncthreads();
    // step 2, cell-level product with the dense matrix; step 3, assembly
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int kk = lane & 3, rw = lane >> 2;
    const int mtn = A.n3p / 8, ksn = A.n3p / 4;
    int cj[NT];                                                  // column of this lane's B element in n-tile j
#pragma unroll
    for (int j = 0; j < NT; ++j) cj[j] = dense_col<VC>(kk, 8 * j + rw);
    for (int mt = warp; mt < mtn; mt += 8) {
        double au[NT][2], ad[NT][2], t1[NT][2], t2[NT][2];       // P Xu + M1 Xd,  M1 Xu + Q Xd,  M2 Xu,  M2 Xd
#pragma unroll
        for (int j = 0; j < NT; ++j) { au[j][0] = au[j][1] = ad[j][0] = ad[j][1] = t1[j][0] = t1[j][1] = t2[j][0] = t2[j][1] = 0.0; }
        const double* m = A.mat + (((long long)e * mtn + mt) * ksn) * 128 + lane;
        const double* mg = A.gk + ((long long)mt * ksn) * 32 + lane;
#pragma unroll 4
        for (int ks = 0; ks < ksn; ++ks) {
            const double mp = __ldg(m + ks * 128), mq = __ldg(m + ks * 128 + 32), m1 = __ldg(m + ks * 128 + 64), m2 = __ldg(m + ks * 128 + 96);
            double gp = 0.0, gn = 0.0;
            if (KPT) { gp = __ldg(mg + ks * 32); gn = -gp; }
            const double* bu = Xu + (size_t)(ks * 4 + kk) * LDW;
            const double* bd = Xd + (size_t)(ks * 4 + kk) * LDW;
#pragma unroll
            for (int j = 0; j < NT; ++j) {
                const double xu = bu[cj[j]], xd = bd[cj[j]];
                dense_dmma(au[j][0], au[j][1], mp, xu); dense_dmma(au[j][0], au[j][1], m1, xd);
                dense_dmma(ad[j][0], ad[j][1], m1, xu); dense_dmma(ad[j][0], ad[j][1], mq, xd);
                dense_dmma(t1[j][0], t1[j][1], m2, xu); dense_dmma(t2[j][0], t2[j][1], m2, xd);
                if (KPT) { dense_dmma(t2[j][0], t2[j][1], gp, xu); dense_dmma(t1[j][0], t1[j][1], gn, xd); }
            }
        }
        const int g = node[mt * 8 + rw];
        if (g < 0) continue;
#pragma unroll
        for (int j = 0; j < NT; ++j) {
            const int v = v0 + 4 * j + kk;
            if (v >= A.nvec) continue;
            // Yu = Au - i T2,  Yd = Ad + i T1
            double* yu = A.Y + ((2LL * g) * A.ldy + v) * 2;
            double* yd = A.Y + ((2LL * g + 1) * A.ldy + v) * 2;
            const double ur = au[j][0] + t2[j][1], ui = au[j][1] - t2[j][0], dr = ad[j][0] - t1[j][1], di = ad[j][1] + t1[j][0];
            atomicAdd(yu, A.fr * ur - A.fi * ui); atomicAdd(yu + 1, A.fr * ui + A.fi * ur);
            atomicAdd(yd, A.fr * dr - A.fi * di); atomicAdd(yd + 1, A.fr * di + A.fi * dr);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// step 4 of P:551-561, the nonlocal part, as separate kernels (the column kernel fuses the expansion; here the local part
// is a different kernel). The coefficients C = P~^T X come from proj_gather_kernel (csf_kernels.cuh).

// D = Delta C per atom, plain layout [crows][ldc] complex (row = atom_coff + 2 chi + spin), eq.76
struct DeltaPlainParams {
    const double2* C; double2* D; long long ldc; int nvec;
    const double2* C2;            // NULL, or the gather with Im P~: the coefficients are C - i C2 = (Re P~ + i Im P~)^+ X
    double fr, fi;                // D = f Delta C
    const long long* atom_coff; const int* atom_npj; const int* atom_type;
    const double2* delta; const long long* delta_ptr;
};

__global__ void __launch_bounds__(256) delta_plain_kernel(const __grid_constant__ DeltaPlainParams A) {
    const int atom = blockIdx.x;
    const int v = blockIdx.y * 32 + (threadIdx.x & 31);
    const int nr = 2 * A.atom_npj[atom];
    const double2* Dl = A.delta + A.delta_ptr[A.atom_type[atom]];
    const long long base = A.atom_coff[atom];
    if (v >= A.nvec) return;
    for (int r = threadIdx.x >> 5; r < nr; r += 8) {
        double sr = 0.0, si = 0.0;
        for (int q = 0; q < nr; ++q) {
            const double2 d = __ldg(Dl + (long long)r * nr + q);
            double2 c = A.C[(base + q) * A.ldc + v];
            if (A.C2) { const double2 c2 = A.C2[(base + q) * A.ldc + v]; c.x += c2.y; c.y -= c2.x; }
            sr = fma(d.x, c.x, sr); sr = fma(-d.y, c.y, sr);
            si = fma(d.x, c.y, si); si = fma(d.y, c.x, si);
        }
        A.D[(base + r) * A.ldc + v] = make_double2(A.fr * sr - A.fi * si, A.fr * si + A.fi * sr);
    }
}

// Y[2 I + spin][v] += sum_chi P~[I, chi] D[atom; 2 chi + spin][v] over the entries (atom, node I) of one gather block;
// P~ is read from g_pack, the fragment-ordered copy the gather kernel uses: [k-step of 4 entries][MT][(chi % 8) * 4 + entry % 4]
struct ExpandPlainParams {
    const double2* D; long long ldc;
    double* Y; long long ldy; int nvec, mt;
    const int* gb_atom; const int* gb_beg; const int* gb_end; const int* gb_k0;
    const int* ent_node; const double* g_pack;
    const double* g_pack_im;      // CPLX: Im P~ in the same order
    const long long* atom_coff; const int* atom_npj;
};

// grid (gather blocks, tiles of 32 vectors), 8 warps, lane = vector. D of the atom for these 32 vectors is staged in shared
// memory once; a warp takes four entries at a time (one k-step of g_pack: the four P~ values of a projector are 32 consecutive bytes)
template <bool CPLX>
__global__ void __launch_bounds__(256) expand_plain_kernel(const __grid_constant__ ExpandPlainParams A) {
    __shared__ double2 Ds[64][32];
    const int b = blockIdx.x, atom = A.gb_atom[b], beg = A.gb_beg[b], end = A.gb_end[b], k0 = A.gb_k0[b];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int v = blockIdx.y * 32 + lane;
    const int npj = A.atom_npj[atom];
    const long long base = A.atom_coff[atom];
    for (int r = warp; r < 2 * npj; r += 8) Ds[r][lane] = v < A.nvec ? A.D[(base + r) * A.ldc + v] : make_double2(0.0, 0.0);
    __syncthreads();
    if (v >= A.nvec) return;
    for (int e = beg + 4 * warp; e < end; e += 32) {
        const double2* pk = reinterpret_cast<const double2*>(A.g_pack + ((long long)(k0 + ((e - beg) >> 2)) * A.mt) * 32);
        double ur[4] = {0.0, 0.0, 0.0, 0.0}, ui[4] = {0.0, 0.0, 0.0, 0.0}, dr[4] = {0.0, 0.0, 0.0, 0.0}, di[4] = {0.0, 0.0, 0.0, 0.0};
        for (int x = 0; x < npj; ++x) {
            const double2 p01 = __ldg(pk + (x >> 3) * 16 + (x & 7) * 2), p23 = __ldg(pk + (x >> 3) * 16 + (x & 7) * 2 + 1);
            const double pv[4] = {p01.x, p01.y, p23.x, p23.y};
            const double2 cu = Ds[2 * x][lane], cd = Ds[2 * x + 1][lane];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                ur[q] = fma(pv[q], cu.x, ur[q]); ui[q] = fma(pv[q], cu.y, ui[q]);
                dr[q] = fma(pv[q], cd.x, dr[q]); di[q] = fma(pv[q], cd.y, di[q]);
            }
            if (CPLX) {                         // + i Im P~ (cu, cd)
                const double2* pki = reinterpret_cast<const double2*>(A.g_pack_im + ((long long)(k0 + ((e - beg) >> 2)) * A.mt) * 32);
                const double2 q01 = __ldg(pki + (x >> 3) * 16 + (x & 7) * 2), q23 = __ldg(pki + (x >> 3) * 16 + (x & 7) * 2 + 1);
                const double pw[4] = {q01.x, q01.y, q23.x, q23.y};
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    ur[q] = fma(-pw[q], cu.y, ur[q]); ui[q] = fma(pw[q], cu.x, ui[q]);
                    dr[q] = fma(-pw[q], cd.y, dr[q]); di[q] = fma(pw[q], cd.x, di[q]);
                }
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (e + q >= end) break;
            const long long I = A.ent_node[e + q];
            double* yu = A.Y + ((2 * I) * A.ldy + v) * 2;
            double* yd = A.Y + ((2 * I + 1) * A.ldy + v) * 2;
            atomicAdd(yu, ur[q]); atomicAdd(yu + 1, ui[q]); atomicAdd(yd, dr[q]); atomicAdd(yd + 1, di[q]);
        }
    }
}

// dst += alpha src on complex128 blocks (the shift term -f c X of a recurrence step on the dense path)
__global__ void __launch_bounds__(256) caxpy_kernel(const double2* __restrict__ src, long long ld, double2* __restrict__ dst, long long ld_dst,
                                                    long long rows, int nvec, double ar, double ai) {
    const long long total = rows * nvec;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long r = t / nvec; const int v = (int)(t % nvec);
        const double2 z = src[r * ld + v];
        double2 o = dst[r * ld_dst + v];
        o.x += ar * z.x - ai * z.y; o.y += ar * z.y + ai * z.x;
        dst[r * ld_dst + v] = o;
    }
}

}  // namespace csf
