// csf_subspace.cuh — kernels of the subspace steps around the filter:
//   gram_kernel       G = A^T B over all spinor rows, A and B viewed as REAL [rows][2N] matrices (re / im interleaved): the four
//                     real products of the complex projection X^dagger Y (eq.71) in one FP64 tensor-core GEMM
//                     (mma.sync m8n8k4 = DMMA), split over row ranges, RED-added into G
//   gram_finish       Hs[m][n] = (G[2m][2n] + G[2m+1][2n+1]) + i (G[2m][2n+1] - G[2m+1][2n]), upper triangle mirrored
//   qtilde_kernel     the real 2N x 2N image of the complex N x N matrix Q
//   rotate_kernel     U = X Q (eq.72) as the real GEMM [rows][2N] x [2N][2N]
//   density_kernel    rho, m at the nodes from a block (eq.4-5), one warp per node
//   Lanczos vector kernels
// This path is a dense contraction (8 N^2 flops per spinor row against 32 N bytes): FP64 tensor-pipe bound.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace csf {

__device__ __forceinline__ void sub_dmma(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
// 16-byte asynchronous copy global -> shared; bytes = 0 zero-fills (rows / columns past the end)
__device__ __forceinline__ void sub_cp16(void* smem_dst, const void* gsrc, int bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc), "r"(bytes) : "memory");
}
__device__ __forceinline__ void sub_cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void sub_cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

constexpr int kGT = 64;            // output tile edge (real columns) of gram / rotate
constexpr int kGK = 32;            // rows (gram) / inner columns (rotate) per shared-memory slab
constexpr int kGP = kGT + 4;       // padded row of a [k][64] slab: a DMMA fragment reads rows k .. k+3 at columns c .. c+7; with the rows 4 doubles
                                   // apart mod 16 each half-warp covers 16 different 8-byte banks (2 wavefronts per LDS.64, the minimum)
constexpr int kRP = kGK + 4;       // padded row of a [64][k] slab (rotate's A operand)
constexpr size_t kGramSmem = (size_t)2 * 2 * kGK * kGP * sizeof(double);
constexpr size_t kRotSmem = (size_t)2 * (kGT * kRP + kGK * kGP) * sizeof(double);

// G[ca][cb] += sum_{r in this CTA's row range} A[r][ca] B[r][cb]; blockIdx.x = (tile m, tile n), blockIdx.y = row range.
// sym: only tiles with n >= m (Hermitian result). 8 warps as 4 x 2: warp (wm, wn) owns the 16 x 32 block at (16 wm, 32 wn) of the
// 64 x 64 tile: 2 A + 4 B fragment loads per 8 DMMAs (an 8 x 64 strip per warp takes 9, and the loads, not the tensor pipe, bound it).
__global__ void __launch_bounds__(256) gram_kernel(const double* __restrict__ A, long long lda, const double* __restrict__ B, long long ldb,
                                                   int ncols, long long rows, long long rows_per_cta, double* __restrict__ G, int ldg, int sym) {
    extern __shared__ __align__(16) double sm[];
    const int ntile = (ncols + kGT - 1) / kGT;
    const int tm = blockIdx.x / ntile, tn = blockIdx.x % ntile;
    if (sym && tn < tm) return;
    const long long r0 = (long long)blockIdx.y * rows_per_cta, r1 = min(rows, r0 + rows_per_cta);
    if (r0 >= r1) return;
    double* As = sm;                                  // [2][kGK][kGP]
    double* Bs = sm + 2 * kGK * kGP;
    const int tid = threadIdx.x, warp = tid >> 5, t = tid & 31;
    const int m0 = tm * kGT, n0 = tn * kGT;
    auto load_slab = [&](int buf, long long rs) {
        // 32 rows x 64 doubles = 1024 16-byte pieces per operand, 4 per thread
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int piece = tid + 256 * q, rr = piece >> 5, cc = (piece & 31) * 2;
            const long long row = rs + rr;
            const bool ra = row < r1;
            sub_cp16(As + (buf * kGK + rr) * kGP + cc, A + (ra ? row : r0) * lda + min(m0 + cc, ncols - 2), (ra && m0 + cc < ncols) ? 16 : 0);
            sub_cp16(Bs + (buf * kGK + rr) * kGP + cc, B + (ra ? row : r0) * ldb + min(n0 + cc, ncols - 2), (ra && n0 + cc < ncols) ? 16 : 0);
        }
        sub_cp_commit();
    };
    const int wm = warp >> 1, wn = warp & 1;
    double c[2][4][2];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) { c[mt][nt][0] = 0.0; c[mt][nt][1] = 0.0; }
    const long long nslab = (r1 - r0 + kGK - 1) / kGK;
    load_slab(0, r0);
    for (long long s = 0; s < nslab; ++s) {
        const int buf = (int)(s & 1);
        if (s + 1 < nslab) { load_slab(buf ^ 1, r0 + (s + 1) * kGK); sub_cp_wait<1>(); } else sub_cp_wait<0>();
        __syncthreads();
        const double* as = As + buf * kGK * kGP + 16 * wm + (t >> 2);
        const double* bs = Bs + buf * kGK * kGP + 32 * wn + (t >> 2);
#pragma unroll
        for (int kk = 0; kk < kGK / 4; ++kk) {
            const double a0 = as[(kk * 4 + (t & 3)) * kGP], a1 = as[(kk * 4 + (t & 3)) * kGP + 8];
#pragma unroll
            for (int nt = 0; nt < 4; ++nt) {
                const double b = bs[(kk * 4 + (t & 3)) * kGP + 8 * nt];
                sub_dmma(c[0][nt][0], c[0][nt][1], a0, b); sub_dmma(c[1][nt][0], c[1][nt][1], a1, b);
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
        const int gm = m0 + 16 * wm + 8 * mt + (t >> 2);
        if (gm >= ncols) continue;
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) {
            const int gn = n0 + 32 * wn + 8 * nt + 2 * (t & 3);
            if (gn < ncols) { atomicAdd(G + (long long)gm * ldg + gn, c[mt][nt][0]); atomicAdd(G + (long long)gm * ldg + gn + 1, c[mt][nt][1]); }
        }
    }
}

// complex N x N result from the real 2N x 2N Gram matrix; sym: the upper triangle decides, the lower is its conjugate
__global__ void __launch_bounds__(256) gram_finish_kernel(const double* __restrict__ G, int ldg, int n, double2* __restrict__ H, int ldh, int sym) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n * n) return;
    const int m = idx / n, q = idx % n;
    const int a = (sym && q < m) ? q : m, b = (sym && q < m) ? m : q;
    const double* g = G + (long long)(2 * a) * ldg + 2 * b;
    double re = g[0] + g[ldg + 1], im = g[1] - g[ldg];
    if (sym && q < m) im = -im;
    if (sym && q == m) im = 0.0;
    H[(long long)m * ldh + q] = make_double2(re, im);
}

// Qt[2m+a][2n+b]: the real matrix of x -> x Q on interleaved (re, im) rows: [[Qr, Qi], [-Qi, Qr]]
__global__ void __launch_bounds__(256) qtilde_kernel(const double2* __restrict__ Q, int ldq, int n, double* __restrict__ Qt, int ldt) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n * n) return;
    const int m = idx / n, q = idx % n;
    const double2 z = Q[(long long)m * ldq + q];
    double* o = Qt + (long long)(2 * m) * ldt + 2 * q;
    o[0] = z.x; o[1] = z.y; o[ldt] = -z.y; o[ldt + 1] = z.x;
}

// U[r][:] = X[r][:] Qt  (real [rows][k2] x [k2][k2]); blockIdx.x = (row tile of 64, column tile), column tile fastest: the
// column tiles of a row tile run together and share its rows in L2
__global__ void __launch_bounds__(256) rotate_kernel(const double* __restrict__ X, long long ldx, const double* __restrict__ Qt, int ldt, int k2,
                                                     double* __restrict__ U, long long ldu, long long rows) {
    extern __shared__ __align__(16) double sm[];
    double* Xs = sm;                                   // [2][kGT][kRP]
    double* Qs = sm + 2 * kGT * kRP;                   // [2][kGK][kGP]
    const int tid = threadIdx.x, warp = tid >> 5, t = tid & 31;
    const int nct = (k2 + kGT - 1) / kGT;
    const int n0 = (int)(blockIdx.x % nct) * kGT;
    const long long r0 = (long long)(blockIdx.x / nct) * kGT;
    auto load_slab = [&](int buf, int k0) {
        // X: 64 rows x 32 doubles = 1024 pieces; Qt: 32 rows x 64 doubles = 1024 pieces; 4 + 4 per thread
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int piece = tid + 256 * q;
            { const int rr = piece >> 4, cc = (piece & 15) * 2; const long long row = r0 + rr; const bool ok = row < rows && k0 + cc < k2;
              sub_cp16(Xs + (buf * kGT + rr) * kRP + cc, X + (row < rows ? row : 0) * ldx + min(k0 + cc, k2 - 2), ok ? 16 : 0); }
            { const int rr = piece >> 5, cc = (piece & 31) * 2; const bool ok = k0 + rr < k2 && n0 + cc < k2;
              sub_cp16(Qs + (buf * kGK + rr) * kGP + cc, Qt + (long long)min(k0 + rr, k2 - 1) * ldt + min(n0 + cc, k2 - 2), ok ? 16 : 0); }
        }
        sub_cp_commit();
    };
    const int wm = warp >> 1, wn = warp & 1;          // warp block 16 x 32, as in gram_kernel
    double c[2][4][2];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) { c[mt][nt][0] = 0.0; c[mt][nt][1] = 0.0; }
    const int nslab = (k2 + kGK - 1) / kGK;
    load_slab(0, 0);
    for (int s = 0; s < nslab; ++s) {
        const int buf = s & 1;
        if (s + 1 < nslab) { load_slab(buf ^ 1, (s + 1) * kGK); sub_cp_wait<1>(); } else sub_cp_wait<0>();
        __syncthreads();
        const double* xs = Xs + (buf * kGT + 16 * wm + (t >> 2)) * kRP + (t & 3);
        const double* qs = Qs + buf * kGK * kGP + 32 * wn + (t >> 2);
#pragma unroll
        for (int kk = 0; kk < kGK / 4; ++kk) {
            const double a0 = xs[kk * 4], a1 = xs[8 * kRP + kk * 4];
#pragma unroll
            for (int nt = 0; nt < 4; ++nt) {
                const double b = qs[(kk * 4 + (t & 3)) * kGP + 8 * nt];
                sub_dmma(c[0][nt][0], c[0][nt][1], a0, b); sub_dmma(c[1][nt][0], c[1][nt][1], a1, b);
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
        const long long row = r0 + 16 * wm + 8 * mt + (t >> 2);
        if (row >= rows) continue;
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) {
            const int gn = n0 + 32 * wn + 8 * nt + 2 * (t & 3);
            if (gn < k2) *reinterpret_cast<double2*>(U + row * ldu + gn) = make_double2(c[mt][nt][0], c[mt][nt][1]);
        }
    }
}

// rho_I, m_I (eq.4-5) of node I: one warp per node, lanes over the vectors; psi = x / sqrt(m_I), so everything is divided by m_I
__global__ void __launch_bounds__(256) density_kernel(const double2* __restrict__ X, long long ld, int nvec, const double* __restrict__ occ,
                                                      const double* __restrict__ inv_mass, long long M, double* __restrict__ out, int accumulate) {
    const long long node = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (node >= M) return;
    const int t = threadIdx.x & 31;
    const double2* xu = X + 2 * node * ld; const double2* xd = xu + ld;
    double r = 0.0, mx = 0.0, my = 0.0, mz = 0.0;
    for (int v = t; v < nvec; v += 32) {
        const double2 u = xu[v], d = xd[v]; const double f = occ[v];
        const double uu = u.x * u.x + u.y * u.y, dd = d.x * d.x + d.y * d.y;
        r = fma(f, uu + dd, r); mz = fma(f, uu - dd, mz);
        mx = fma(2.0 * f, u.x * d.x + u.y * d.y, mx);          // 2 Re(conj(u) d)
        my = fma(2.0 * f, u.x * d.y - u.y * d.x, my);          // 2 Im(conj(u) d)
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        r += __shfl_xor_sync(0xffffffffu, r, o); mx += __shfl_xor_sync(0xffffffffu, mx, o);
        my += __shfl_xor_sync(0xffffffffu, my, o); mz += __shfl_xor_sync(0xffffffffu, mz, o);
    }
    if (t == 0) {
        const double s = inv_mass[node]; double* o = out + 4 * node;
        if (accumulate) { o[0] += s * r; o[1] += s * mx; o[2] += s * my; o[3] += s * mz; }
        else { o[0] = s * r; o[1] = s * mx; o[2] = s * my; o[3] = s * mz; }
    }
}

// ---- Lanczos vector kernels (complex128 vectors of length n; scalars reduced into scratch[0..1] by RED)
// w -= beta vprev;  scratch[0] += Re <v, w>
__global__ void __launch_bounds__(256) lanczos_a_kernel(double2* __restrict__ w, const double2* __restrict__ vprev, const double2* __restrict__ v, double beta, long long n, double* scratch) {
    double s = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        double2 x = w[i]; const double2 p = vprev[i], q = v[i];
        x.x = fma(-beta, p.x, x.x); x.y = fma(-beta, p.y, x.y); w[i] = x;
        s = fma(q.x, x.x, fma(q.y, x.y, s));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(scratch, s);
}
// w -= alpha v;  scratch[1] += |w|^2
__global__ void __launch_bounds__(256) lanczos_b_kernel(double2* __restrict__ w, const double2* __restrict__ v, double alpha, long long n, double* scratch) {
    double s = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        double2 x = w[i]; const double2 q = v[i];
        x.x = fma(-alpha, q.x, x.x); x.y = fma(-alpha, q.y, x.y); w[i] = x;
        s = fma(x.x, x.x, fma(x.y, x.y, s));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(scratch + 1, s);
}
// vprev = v; v = scale * w     (also used for the start: v = v0 / |v0| with w = v0)
__global__ void __launch_bounds__(256) lanczos_c_kernel(double2* __restrict__ vprev, double2* __restrict__ v, const double2* __restrict__ w, double scale, long long n) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        vprev[i] = v[i]; const double2 x = w[i]; v[i] = make_double2(scale * x.x, scale * x.y);
    }
}

}  // namespace csf
