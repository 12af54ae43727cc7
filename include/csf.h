/*
 * csf.h — C ABI of libcsf: Chebyshev-filtered spinor H.X on one NVIDIA B200 (sm_100a).
 *
 * The library computes, for a block X of two-component complex spinor wavefunctions,
 *
 *      Y = T_m(H~) X,   H~ = (Hhat - c I)/e,  c = (a+b)/2,  e = (b-a)/2,
 *      Hhat = M_D^{-1/2} (H^loc + H^nloc) M_D^{-1/2}
 *
 * where H^loc, H^nloc are the finite-element discretised local and nonlocal (spin-orbit
 * pseudopotential) parts of the noncollinear Kohn-Sham Hamiltonian of arxiv 2410.02754 and M_D is the
 * GLL-lumped (diagonal) mass matrix. Citations "P:<line>" are lines of the paper text:
 *
 *   spinor coefficients U_{2I+alpha,n}, alpha = 0 (up), 1 (down)                     P:290-302 eq.38-39
 *   H^loc_{2I+a,2J+b} = int [1/2 grad N_I . grad N_J + V_eff N_I N_J] d_ab
 *                        + sum_d B^d N_I N_J sigma^d_ab          (Gamma point, k = 0)  P:304 eq.40, eq.16
 *   H^nloc_{2I+a,2J+b} = sum_atoms sum_{X X'} P_{I X} D^{X X'}_{ab} conj(P_{J X'})     P:308 eq.41, eq.14
 *   Delta_{2X+a,2X'+b} = D^{X X'}_{ab}                                                P:517-519 eq.76
 *   cell-level evaluation: extract X^(e) = R^(e) X, apply H^(e), assemble sum_e R^(e)T Y^(e)
 *                                                                                     P:507 eq.74, eq.84
 *   M diagonal through GLL quadrature at the FE nodes; filter built on M^-1 H
 *   T_{k+1}(H~) = 2 H~ T_k(H~) - T_{k-1}(H~), unwanted spectrum [a,b] -> [-1,1]        P:463-469 eq.70
 *
 * Readings where the paper is silent: the similarity-equivalent Hermitian form
 * M_D^{-1/2} H M_D^{-1/2} is used (X and Y live in the Loewdin-scaled basis); T_m is the plain first-kind
 * Chebyshev polynomial; the stiffness integral is exact; V_eff and B are collocated at the GLL nodes;
 * projector entries P_{I X} are supplied already integrated; nodes on a Dirichlet face are removed.
 *
 * Conventions
 *   - Every function returns CSF_OK (0) or a negative error code; nothing throws or aborts across the ABI.
 *     csf_last_error() gives a text for the last failure on that context.
 *   - "host" pointers are ordinary CPU memory, copied before the call returns (the caller may free them).
 *     "device" pointers are CUDA device memory on the context's device, owned by the caller.
 *   - Device multivector layout: element (node I, spin alpha, vector n) is the complex128 at
 *     d[(2*I + alpha)*ld + n], ld >= nvec  (row 2I+alpha as in P:302; vector index fastest).
 *   - Node numbering is the library's: unconstrained nodes only, x fastest, then y, then z; use
 *     csf_node_coords() instead of guessing.
 *   - csf_apply_H and csf_filter only ENQUEUE work on the context's stream and return without
 *     synchronising; create/set_* /destroy may synchronise.
 *   - There is no CPU fallback: without a CUDA device every compute entry point fails with CSF_ECUDA.
 */
#ifndef CSF_H
#define CSF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct csf_ctx csf_ctx;                 /* opaque; owns all device-side operator tables */
typedef struct { double re, im; } csf_c128;     /* layout-compatible with cuDoubleComplex / torch.complex128 */

enum { CSF_OK = 0, CSF_EINVAL = -1, CSF_ENOMEM = -2, CSF_ECUDA = -3, CSF_ESTATE = -4, CSF_EUNSUPPORTED = -5 };
enum { CSF_BC_PERIODIC = 0, CSF_BC_DIRICHLET = 1, CSF_BC_FREE = 2 /* natural BC: not supported on the GPU path */ };
enum { CSF_FP64 = 0, CSF_FP32_INTERMEDIATE = 1 };

/* Create the mesh, cells and GLL nodes: an axis-aligned box of `box` bohr meshed by
 * ncell[0] x ncell[1] x ncell[2] congruent hexahedral cells carrying tensor-product Lagrange bases of
 * degree `order` (1..7) on GLL nodes; bc[d] is CSF_BC_PERIODIC or CSF_BC_DIRICHLET per direction.
 * `device` is the CUDA ordinal; `cuda_stream` is a cudaStream_t (borrowed, may be NULL = default stream)
 * on which all later work is enqueued. All arrays are host pointers. Errors: CSF_EINVAL (bad argument),
 * CSF_EUNSUPPORTED (CSF_BC_FREE, order > 7), CSF_ECUDA, CSF_ENOMEM. */
int csf_create(csf_ctx** out, const int ncell[3], const double box[3], int order, const int bc[3],
               int device, void* cuda_stream);

/* Free the context and every device table it owns. NULL is accepted. */
int csf_destroy(csf_ctx* ctx);

/* Rebind the stream later work is enqueued on (borrowed cudaStream_t). */
int csf_set_stream(csf_ctx* ctx, void* cuda_stream);

/* M = number of unconstrained FE nodes per spin component ("M^{h,p}"); a spinor block has 2M rows. */
int csf_num_nodes(const csf_ctx* ctx, int64_t* M);

/* GLL node positions in the library's numbering, host array [M][3] (bohr). A periodic node is reported
 * at its image inside [0, box). */
int csf_node_coords(const csf_ctx* ctx, double* xyz_host);

/* Lumped GLL mass m_I = sum_e J^(e) w_i w_j w_k (eq.43 under GLL quadrature), host array [M]. */
int csf_mass_diag(const csf_ctx* ctx, double* m_host);

/* Set the spin potential at the nodes (eq.16, eq.40): veff host [M] (Ha), bxyz host [M][3]
 * (B_xc components; NULL means B = 0). Node I contributes the block m_I (V_I I_2 + B_I . sigma). */
int csf_set_potential(csf_ctx* ctx, const double* veff, const double* bxyz);

/* Set the atom-centred projectors and the spin-coupled D matrices (eq.41-42, eq.76).
 *   natoms           number of atoms; 0 clears the nonlocal part (all other pointers may then be NULL)
 *   node_ptr         host [natoms+1]: atom a's support rows are node_idx[node_ptr[a] .. node_ptr[a+1])
 *   node_idx         host: global node ids (0 <= id < M), no duplicates within one atom
 *   nproj            host [natoms]: n_pj of each atom (scalar projector columns, spin-diagonal as in eq.78)
 *   pvals            host: atom a's block [n_a][nproj[a]] row-major, blocks concatenated; entry = P_{I X},
 *                    the already integrated value of eq.42 at k = 0 (real)
 *   atom_type        host [natoms]: index gamma_a into the Delta tables
 *   ntypes, delta, delta_ptr
 *                    type t owns delta[delta_ptr[t] .. delta_ptr[t+1]) = [(2 npj)][(2 npj)] row-major with
 *                    composite index 2X+alpha (eq.76); must be Hermitian for a Hermitian H (not checked)
 * Errors: CSF_EINVAL on inconsistent sizes or out-of-range ids. */
int csf_set_projectors(csf_ctx* ctx, int natoms, const int64_t* node_ptr, const int64_t* node_idx,
                       const int* nproj, const double* pvals, const int* atom_type, int ntypes,
                       const csf_c128* delta, const int64_t* delta_ptr);

/* Bytes of device workspace csf_apply_H / csf_filter need for blocks of up to nvec vectors in `mode`. */
int csf_workspace_bytes(const csf_ctx* ctx, int nvec, int mode, size_t* bytes);

/* Y = Hhat X (one application of M_D^{-1/2} H M_D^{-1/2}; P:551-561 steps 2-4). dX, dY: device, [2M][ld]
 * complex128, dY must not alias dX. d_work: device, >= csf_workspace_bytes(nvec, CSF_FP64). Enqueues only.
 * Errors: CSF_ESTATE if the potential was never set, CSF_EINVAL on NULL / ld < nvec / nvec < 0 /
 * too small workspace, CSF_ECUDA. nvec = 0 is a no-op. */
int csf_apply_H(csf_ctx* ctx, const csf_c128* dX, csf_c128* dY, int64_t ld, int nvec,
                void* d_work, size_t work_bytes);

/* csf_apply_H for callers that may not allocate (CUDA graph capture, tight serving loops): the same launch sequence,
 * with the projector-coefficient scratch (C = P~^T X and C~ = Delta C of P:551-561 steps 3-4) in an array of
 * CSF_STATIC_SCRATCH_BYTES that is part of the library image: every GPU that loads libcsf.so holds it until the process
 * exits. The call takes no workspace and calls no cudaMalloc / cudaFree / allocating library routine; the scratch is
 * cleared by the call itself (it keeps the previous call's contents otherwise). ALL contexts and calls on one device
 * share the array: two calls that overlap on the GPU (different streams, no dependency) race; order them.
 * Errors: as csf_apply_H, plus CSF_EUNSUPPORTED with a text naming both sizes when the scratch for (this context's
 * projectors, nvec) exceeds CSF_STATIC_SCRATCH_BYTES, CSF_ESTATE while per-kernel profiling is enabled (it creates
 * events), CSF_ECUDA if the array's device address cannot be resolved. Without projectors no scratch is used. */
#define CSF_STATIC_SCRATCH_BYTES (8u << 20)
int csf_apply_H_static(csf_ctx* ctx, const csf_c128* dX, csf_c128* dY, int64_t ld, int nvec);

/* Y = T_degree((Hhat - c)/e) X with c = (a+b)/2, e = (b-a)/2 (eq.70). degree = 0 copies X to Y.
 * Same pointer rules as csf_apply_H; X is not modified. mode: CSF_FP64, or CSF_FP32_INTERMEDIATE (complex128
 * in and out; both recurrence buffers complex64 and the cell-level arithmetic FP32 in between, projector coefficients
 * kept in FP64; agrees with the FP64 result to about 1e-5 relative).
 * Errors: CSF_EINVAL also for degree < 0 or a >= b. Enqueues only. */
int csf_filter(csf_ctx* ctx, const csf_c128* dX, csf_c128* dY, int64_t ld, int nvec,
               int degree, double a, double b, int mode, void* d_work, size_t work_bytes);

/* Same operation with HOST buffers hX, hY ([2M][ld] complex128, pinned or pageable): the library stages
 * column chunks through device memory it allocates itself (host->device copy, filter, device->host copy)
 * and SYNCHRONISES before returning. This is the end-to-end entry point. */
int csf_filter_host(csf_ctx* ctx, const csf_c128* hX, csf_c128* hY, int64_t ld, int nvec,
                    int degree, double a, double b, int mode);

/* Columns per staged chunk of csf_filter_host (default 64; >= 1). */
int csf_set_host_chunk(csf_ctx* ctx, int ncols);

/* Per-kernel CUDA-event timing. While enabled, every kernel the context launches is bracketed by two events
 * on the context's stream. csf_profile_read SYNCHRONISES the stream, returns the summed device time (ms) and the
 * number of launches of `kind` since the last read, and clears that kind. kind: CSF_KIND_CELL (gather -> cell-level
 * local apply -> assembly and recurrence update, a1-a4, a7, a8), CSF_KIND_PGATHER (a5), CSF_KIND_DELTA (a6),
 * CSF_KIND_AUX (block copy / zero). */
enum { CSF_KIND_CELL = 0, CSF_KIND_PGATHER = 1, CSF_KIND_DELTA = 2, CSF_KIND_AUX = 3, CSF_NKINDS = 4 };
int csf_profile_enable(csf_ctx* ctx, int on);
int csf_profile_read(csf_ctx* ctx, int kind, double* ms_total, int64_t* launches);

/* Measure the FP64 arithmetic peaks of `device` with register-resident loops (no memory traffic): tflops_fma from
 * independent DFMA chains, tflops_mma from mma.sync m8n8k4 f64 (DMMA) chains. Synchronises. Either pointer may be NULL. */
int csf_probe_fp64_peak(int device, double* tflops_fma, double* tflops_mma);

/* The same two loops side by side (even warps DFMA chains, odd warps DMMA chains): *tflops_total is the sum of both.
 * On B200 it equals either loop alone (36.4 TF/s against 33.9 / 36.7): DFMA and DMMA issue to the same FP64 units, so the
 * FP64 roofline has ONE peak and tensor-core tiles buy no extra rate. Synchronises. */
int csf_probe_fp64_mixed(int device, double* tflops_total);

/* Which column-kernel variant a block of nvec vectors runs with in `mode` on this context: *lanes = 32 (orders 4 and 5:
 * 8 vectors per CTA) or 16 (the other orders: 4 vectors per CTA; 8 lanes = 2 vectors at order 7). Environment variables read
 * by csf_create pin the variant for the parity tests, which run every case through each kernel: CSF_LANES=16 (the 16-lane
 * kernel at orders 4 and 5 too), CSF_KERNEL=ws (the warp-specialised streaming kernel of csf_colws.cuh, orders 4 and 5;
 * parity-green but slower). Host-only query. */
int csf_column_lanes(const csf_ctx* ctx, int nvec, int mode, int* lanes);

/* Whether csf_filter runs a block of nvec vectors in `mode` on its fused half-block path (*fused = 1) or with one projector
 * gather kernel per recurrence step (*fused = 0). Fused path (eq.84: the inner sum C^a = P^{a,T} X^(e') is all that a
 * step needs from the other cells): complex128, order 5, 8 vectors per CTA, 18 projectors per atom, a multiple of 64 vectors. The block is
 * split into two halves (the first a multiple of 8 vectors) whose column steps alternate, and every column launch computes, in
 * two extra warps, the projector coefficients the OTHER half needs next: the HBM-bound gather runs beside the latency-bound
 * column step instead of after it. Results differ from the unfused path by summation order only.
 * CSF_FUSED_GATHER=0 | 1 (read by csf_create) switches the path off | on for every block of >= 9 vectors (parity tests).
 * Host-only query. */
int csf_filter_fused_gather(const csf_ctx* ctx, int nvec, int mode, int* fused);

/* Number of kernel launches (own kernels only, memsets excluded) enqueued by this context so far. */
int csf_launch_count(const csf_ctx* ctx, int64_t* launches);

/* Select a kernel variant: 0 = library default; 1 = always take the general (predicated) column kernel, also on
 * fully periodic meshes where the predicate-free specialisation would be chosen (test hook). CSF_EINVAL if unknown. */
int csf_set_variant(csf_ctx* ctx, int variant);

/* Test / tuning hook for the traversal of the column kernels (no effect on results beyond summation order): seg_len =
 * cells of a (cx, cy) column that one CTA marches through before the z-face is handed over through global memory
 * (0 = the kernel's default: 16, or the whole column up to 64 cells for orders 4 and 5); chunk_group = vector chunks of one
 * column scheduled back to back (>= 1, default 16). The parity tests use it to put segment boundaries, the final carry
 * flush and multi-group grids on small meshes. CSF_EINVAL on seg_len < 0 or chunk_group < 1. */
int csf_set_tuning(csf_ctx* ctx, int seg_len, int chunk_group);

/* ---- Subspace steps around the filter -----------------------------------------------
 * X is a block in the same layout and basis as for csf_filter (Loewdin-scaled: X = M_D^{1/2} U), so the generalized problem
 * of PAPER.md:473-477 eq.71, X_s^dagger H X_s Q = X_s^dagger M X_s Q Lambda, reads Hs Q = Ss Q Lambda with the two matrices below. */

/* Device workspace of csf_rr_project / csf_rr_rotate for a block of nvec vectors. */
int csf_rr_workspace_bytes(const csf_ctx* ctx, int nvec, size_t* bytes);

/* Rayleigh-Ritz projection (eq.71): dHs = X^dagger Hhat X, dSs = X^dagger X, both DEVICE complex128 [nvec][nvec] row-major,
 * exactly Hermitian (the upper triangle is computed, the lower mirrored). FP64 tensor-core GEMMs over all 2M rows.
 * Enqueues on the context's stream; X is not modified. Errors as csf_apply_H. */
int csf_rr_project(csf_ctx* ctx, const csf_c128* dX, int64_t ld, int nvec, csf_c128* dHs, csf_c128* dSs,
                   void* d_work, size_t work_bytes);

/* Solve the projected problem Hs Q = Ss Q Lambda (eq.71; n x n, dense: cuSOLVER's zhegvd, loaded at first use). dQ: DEVICE
 * [n][n] row-major, column j = eigenvector j with Q^dagger Ss Q = I; lambda_host: HOST [n], ascending. SYNCHRONISES.
 * CSF_EINVAL if Ss is not positive definite (linearly dependent block), CSF_EUNSUPPORTED if libcusolver is missing. */
int csf_rr_solve(csf_ctx* ctx, const csf_c128* dHs, const csf_c128* dSs, int n, csf_c128* dQ, double* lambda_host);

/* Subspace rotation (eq.72): dU = X Q, dU [2M][ldu] must not alias dX; Q as returned by csf_rr_solve (any
 * complex [nvec][nvec] row-major matrix is accepted). Needs csf_rr_workspace_bytes. Enqueues on the stream. */
int csf_rr_rotate(csf_ctx* ctx, const csf_c128* dX, int64_t ld, int nvec, const csf_c128* dQ, csf_c128* dU, int64_t ldu,
                  void* d_work, size_t work_bytes);

/* Electron density and magnetisation at the nodes (eq.4-5) from a block of states with occupations
 * occ_host[nvec] (HOST): psi^alpha_n(r_I) = X[2I+alpha][n] / sqrt(m_I), d_rho_m (DEVICE) [M][4] = rho, m_x, m_y, m_z.
 * accumulate != 0 adds to d_rho_m (blocks of states are summed), else overwrites. Copies occ, then enqueues on the stream. */
int csf_density(csf_ctx* ctx, const csf_c128* dX, int64_t ld, int nvec, const double* occ_host, double* d_rho_m, int accumulate);

/* k steps of the Lanczos recurrence on Hhat on the device (lambda_min, lambda_max from Lanczos), start vector
 * d_v0 (DEVICE complex128 [2M], any non-zero norm; not modified): alpha_host[k], beta_host[k] (HOST) receive the tridiagonal
 * coefficients, beta_host[j] = |w| after step j (beta_host[k-1] is the residual norm), *steps_done <= k the steps taken (an
 * invariant subspace ends the recurrence early). SYNCHRONISES (two scalars come back per step). */
int csf_lanczos_workspace_bytes(const csf_ctx* ctx, size_t* bytes);
int csf_lanczos(csf_ctx* ctx, const csf_c128* d_v0, int k, double* alpha_host, double* beta_host, int* steps_done,
                void* d_work, size_t work_bytes);

/* Smallest and largest eigenvalue of the symmetric tridiagonal matrix (alpha[k], beta[0..k-2]) by Sturm bisection: the Ritz
 * values theta_min, theta_max of a csf_lanczos run; theta_max + beta[k-1] is the customary upper bound b of the filter. Host only. */
int csf_tridiag_extremes(const double* alpha, const double* beta, int k, double* theta_min, double* theta_max);

/* Text of the last error recorded on ctx (never NULL; "" if none). With ctx = NULL: last csf_create failure. */
/* ---- potential on a general quadrature rule, dense cell-matrix form of H X --------------------------
 * PAPER.md:528-547 eq.79-83: V_eff and B are given at the n_q^3 Gauss-Legendre points of every cell (eq.44);
 * the cell-level potential matrices V^(e) = (N~ o (w J v^(e))) N~^T are dense n_p^3 x n_p^3. P:551-561 eq.84: H X is then
 * computed cell by cell: extraction R^(e) X, product with the dense cell-level matrix (kinetic + potential, 2x2 in spin),
 * assembly, plus the nonlocal part. This is the paper's own formulation; csf_apply_H (sum-factorised, nodal potential)
 * is the fast path, and bench.py reports both. */

/* Physical coordinates of the quadrature points, xyz_host[E][nq^3][3], cell e = cx + ncx (cy + ncy cz), point
 * q = qx + nq (qy + nq qz): where the caller evaluates its fields for csf_set_potential_quadrature. 1 <= nq <= 16. */
int csf_quadrature_points(const csf_ctx* ctx, int nq, double* xyz_host);

/* vq_host[E][nq^3][4] = V_eff, B_x, B_y, B_z at those points (host, copied). Builds on the device, for every cell, the four
 * real matrices 1/2 K^(e) + V^(e) +- B_z^(e), B_x^(e), B_y^(e) with the Loewdin scaling applied: 4 (n_p^3)^2 doubles per
 * cell (1.5 MB at order 5). Synchronises. Independent of csf_set_potential; csf_set_projectors applies to both paths.
 * Errors: CSF_EINVAL (NULL, nq out of range), CSF_ENOMEM when the matrices do not fit device memory, CSF_ECUDA. */
int csf_set_potential_quadrature(csf_ctx* ctx, int nq, const double* vq_host);

/* Bytes of device workspace csf_filter_dense needs for nvec vectors (one block buffer + projector coefficients);
 * csf_apply_H_dense is content with the same or less. */
int csf_dense_workspace_bytes(const csf_ctx* ctx, int nvec, size_t* bytes);

/* Y = Hhat X through the dense cell matrices (eq.84). Pointer rules and errors as csf_apply_H; CSF_ESTATE if
 * csf_set_potential_quadrature was never called. Enqueues only. */
int csf_apply_H_dense(csf_ctx* ctx, const csf_c128* dX, csf_c128* dY, int64_t ld, int nvec, void* d_work, size_t work_bytes);

/* csf_filter (eq.70, FP64) with every H apply going through the dense cell matrices: the filter for operators
 * only the dense path holds (general quadrature rule, k-points). Arguments and errors as csf_filter. Enqueues only. */
int csf_filter_dense(csf_ctx* ctx, const csf_c128* dX, csf_c128* dY, int64_t ld, int nvec,
                     int degree, double a, double b, void* d_work, size_t work_bytes);

/* ---- k-point (Bloch) Hamiltonian, on the dense path ------------------------------------------------
 * PAPER.md:147-169 eq.21-24: H^k = e^{-ik.r} H e^{ik.r}; discretised (eq.40, eq.41-42)
 *   H^k,loc  = int [1/2 grad N_I.grad N_J - i N_I k.grad N_J + (|k|^2/2 + V_eff) N_I N_J] d_ab + sum_d B^d N_I N_J sigma^d_ab
 *   H^k,nloc = sum_a sum_{X X'} P^k_{I X} D^{X X'}_ab conj(P^k_{J X'}),  P^k_{I X} complex (Bloch phases e^{-ik.(r - L_q)})
 * The gradient term is integrated exactly; |k|^2/2 is integrated with V_eff's rule (reading A19). The
 * sum-factorised entry points (csf_apply_H, csf_apply_H_static, csf_filter, csf_filter_host) hold the Gamma-point operator
 * with real projectors and fail with CSF_ESTATE while a k-point or complex projectors are set. csf_rr_project and csf_lanczos
 * apply the operator the context holds: in that state Hhat^k through the dense cell matrices (quadrature-rule potential), so
 * that csf_lanczos -> csf_filter_dense -> csf_rr_project / _solve / _rotate -> csf_density is a whole ChFSI pass at a k-point. */

/* Bloch vector k_host[3] (1/bohr); (0, 0, 0) switches the k-point terms off. Invalidates the cell matrices:
 * csf_set_potential_quadrature must be called after it. Meaningful on periodic directions (not checked). */
int csf_set_kpoint(csf_ctx* ctx, const double* k_host);

/* csf_set_projectors with complex entries pvals[...] = P^{a,k}_{I X} of eq.42 (same layout; all host pointers). */
int csf_set_projectors_complex(csf_ctx* ctx, int natoms, const int64_t* node_ptr, const int64_t* node_idx,
                               const int* nproj, const csf_c128* pvals, const int* atom_type, int ntypes,
                               const csf_c128* delta, const int64_t* delta_ptr);

const char* csf_last_error(const csf_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* CSF_H */
