/* ark_m1.h — C ABI of libark_m1.so: the radiative-transfer step of the asymptotic-preserving (AP),
 * well-balanced (WB) M1 scheme of arXiv 2011.13926 (ARK-RT), hand-written CUDA for NVIDIA B200 (sm_100a), fp64.
 *
 * What one handle is: one uniform 2-D grid of nx*ny cells carrying the radiative energy E, the radiative flux
 * F = (Fx, Fy), the absorption and scattering opacities sigma_a, sigma_s (sigma_t = sigma_a + sigma_s) and,
 * optionally, a gas temperature T.  PAPER.md:64-69 (Eq. 3) is the system advanced; PAPER.md:142 the grid.
 *
 * Layout.  Every field is a row-major plane [ny][nx] of doubles, x fastest.  F = [Fx plane | Fy plane]
 * (2*nx*ny doubles).  A solver vector is [E | Fx | Fy] (3*nx*ny doubles).
 *
 * Pointers.  Every `const double*` / `double*` array argument may be a DEVICE pointer (cudaMalloc, e.g. a
 * torch tensor's data_ptr()) or a HOST pointer (pinned or pageable): the library copies with
 * cudaMemcpyAsync(cudaMemcpyDefault) on the handle's stream.  The library never keeps a caller pointer after
 * the call returns: set_* calls copy in (for pageable host memory the copy has completed on return; for pinned
 * or device memory it is ordered on the handle's stream, so the caller must not overwrite the source before
 * that stream reaches it), get_* calls copy out and synchronise the stream before returning.  All device
 * memory the handle allocates is owned by the handle and freed by ark_m1_destroy.
 *
 * Errors.  Functions returning int return 0 (or a non-negative count) on success and a negative ARK_M1_E_*
 * code on failure; ark_m1_last_error(h) then holds a message.  Non-convergence of the linear solver is NOT an
 * error (see ark_m1_step_implicit).  No call ever falls back to a CPU computation.
 *
 * Threading.  A handle is not thread-safe; different handles are independent.
 */
#ifndef ARK_M1_H
#define ARK_M1_H

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define ARK_M1_API __attribute__((visibility("default")))
#else
#define ARK_M1_API
#endif

typedef struct ark_m1 ark_m1; /* opaque */

/* Boundary condition of one side (PAPER.md:142 ghost cells; Eq. 24, for the given-state form). */
enum { ARK_M1_BC_PERIODIC = 0, ARK_M1_BC_DIRICHLET = 1, ARK_M1_BC_OUTFLOW = 2 };
/* Side indices for ark_m1_set_boundary. */
enum { ARK_M1_XLO = 0, ARK_M1_XHI = 1, ARK_M1_YLO = 2, ARK_M1_YHI = 3 };
typedef struct { int xlo, xhi, ylo, yhi; } ark_m1_bc;

/* Error codes. */
enum {
    ARK_M1_OK = 0,
    ARK_M1_E_ARG = -1,      /* bad argument (NULL, dt <= 0, tol <= 0, restart < 1, unknown key, ...) */
    ARK_M1_E_CUDA = -2,     /* a CUDA runtime call failed (message holds cudaGetErrorString) */
    ARK_M1_E_ALLOC = -3,    /* device allocation failed */
    ARK_M1_E_NOTSET = -4,   /* step called before ark_m1_set_state */
    ARK_M1_E_NONFINITE = -5,/* the solver met a non-finite norm (state or opacity holds NaN/Inf) */
    ARK_M1_E_UNSUPPORTED = -6
};

/* Create a solver for an nx*ny grid with cell sizes dx, dy and speed of light c.
 * bc == NULL means periodic on all sides; periodic must be set on both sides of a direction.
 * Uses the current CUDA device (every later call on the handle makes that device current for its duration and restores the
 * caller's) and the legacy default stream until ark_m1_set_stream.  Limits: ny <= 262140 (several kernels map four rows to one
 * gridDim.y slot); grids of 2^31 cells or more run on the generic explicit kernel only.
 * Returns NULL on bad arguments, beyond the limits, or when no CUDA device is usable. */
ARK_M1_API ark_m1* ark_m1_create(int nx, int ny, double dx, double dy, double c, const ark_m1_bc* bc);
ARK_M1_API void    ark_m1_destroy(ark_m1* h);

/* All later work of this handle is enqueued on `cuda_stream` (a cudaStream_t, e.g. torch's current stream). */
ARK_M1_API int ark_m1_set_stream(ark_m1* h, void* cuda_stream);

/* Copy in the state and the opacities (north_star: ark_m1_set_state(E, F, sigma_a, sigma_s[, T])).
 * T == NULL: no emission and no matter coupling (pure radiation, dE/dt + div F = -c sigma_a E).
 * T != NULL: emission c sigma_a a_r T^4 and the matter-energy equation (Eq. 4) are switched on. */
ARK_M1_API int ark_m1_set_state(ark_m1* h, const double* E, const double* F, const double* sigma_a, const double* sigma_s,
                     const double* T);

/* One Dirichlet ghost line on `side` (used only where that side's bc is ARK_M1_BC_DIRICHLET): ny values per
 * array for XLO/XHI, nx values for YLO/YHI; F_g = [Fx line | Fy line].  The ghost cell enters the face fluxes
 * and the WB source exactly like an interior cell (Eq. 24) and is constant in time. */
ARK_M1_API int ark_m1_set_boundary(ark_m1* h, int side, const double* E_g, const double* F_g, const double* sigma_a_g,
                        const double* sigma_s_g);

/* Scheme switches (defaults = the paper's scheme):
 *   "well_balanced" 1: Eqs. 18-19          0: Eq. 16, cell-centred source
 *   "ap_mode"       1: alpha of Eq. 25         0: alpha = 1 (standard HLL)   2: Eq. C.8
 *   "eig_mode"      0: Eq. 14                  1: fixed +-c                  2: fixed +-c/sqrt(3)
 *   "closure"       0: M1 chi(f)                1: P1, chi = 1/3
 *   "linearisation" 0: analytic pressure Jacobian (Newton)   1: frozen Eddington tensor
 *   "eig_floor"     x: lambda+ >= x c, lambda- <= -x c; default 0
 *   "a_r"           radiation constant (default 1)
 *   "orthogonalisation" 1: one-pass classical Gram-Schmidt (default)   2: CGS2 (re-orthogonalise once)
 *   "assembly_kernel"   1: marching assembly for the matrix-free operator (default)   0: tile assembly (always used by operator 0)
 *   "krylov"            0: restarted GMRES(restart) (north_star, default)   1: BiCGStab, the paper's solver,
 *                       right-preconditioned with the same block-Jacobi; `restart` is then ignored and the returned count is in
 *                       BiCGStab iterations (two operator applications each)
 *   "vectors_per_pass"  basis vectors handled per pass of the multi-dot / multi-axpy kernels, 1..16 (default 16, by measurement)
 *   "release_workspace" non-zero: free the implicit workspace (operator planes, Krylov basis, multigrid hierarchy) now; the next
 *                       implicit step allocates what it needs again.  Synchronises.
 *   "kernel_timing"     1: time every kernel launch with CUDA events (see ark_m1_get_kernel_stats); default 0
 *   "explicit_kernel"   0: one-thread-per-cell kernel (generic; all scheme switches)   1: row-marching kernel, 128-column blocks
 *                       3: row-marching kernel, one warp per block, four-slot register rotation (no window copies), closure one
 *                          row ahead of the faces, cp.async row prefetch (default)
 *   "operator"          1: matrix-free coefficient planes, flux form (default: 5% faster per solve at 4096^2)
 *                       0: block stencil (BSR 3x3 on the 5-point graph, pre-multiplied by M^-1)
 *   "arnoldi_block"     columns of the Arnoldi process built per pass over the basis (the iterates and the iteration count are
 *                          GMRES(m)'s in every case; the stop test and the iteration limit act per column):
 *                          5 (default), 4, 3: s-step blocks (W_1 = A M^-1 v_j, W_k = (A M^-1 - 1) W_{k-1}; one dot pass, one update
 *                             pass, Cholesky-based in-block solve — predicted by the dot pass and applied by the update pass for
 *                             well-conditioned blocks, a pass of its own with a second round for ill-conditioned ones —, Hessenberg
 *                             columns recovered on the device); columns a restart length leaves over use the two-column step
 *                          2: two columns per pass     1: one
 *                          applies to GMRES + block-Jacobi + matrix-free operator + one-pass orthogonalisation, restart <= 120
 *   "op_recompute"      what the preconditioned matrix-free operator rebuilds in registers instead of loading it (same operator up
 *                          to rounding; cells with folded neighbours (outflow sides) and clamped cells always use the stored values):
 *                          2 (default): each cell's diagonal block, from J and the four faces' coefficients (3 x 3 solve in place of
 *                             the nine M^-1 planes), and J itself from the cell's reduced flux (2 planes in place of 9):
 *                             136 B per cell per application; needs the default scheme and the marching assembly, else acts as 1
 *                          1: the diagonal block only: 192 B     0: nothing, M^-1 and J are loaded: 264 B
 *   "op_pair"           1 (default): inside an s-step block two applications of the preconditioned operator go through ONE pass over
 *                          the coefficient planes (160 instead of 2 x 136 B per cell) where op_recompute = 2 is in effect (default
 *                          scheme) and the grid is at least 4 x 4 and not a slab of a decomposed grid; two passes otherwise.
 *                          0: always two passes.  Same results.
 *   "apply_operator_precond"  1: ark_m1_apply_operator returns A M^-1 V through the solver's preconditioned kernel (matrix-free
 *                          operator only); 0 (default): A V
 *   "basis_precision"   64 (default) or 32: storage precision of the GMRES Arnoldi basis.  32 = compressed-basis GMRES: the basis
 *                       vectors are stored in single precision, every computation (operator, dots, updates, Hessenberg,
 *                       solution, true residual at each restart) stays fp64 and the solve ends at the same fp64 tolerance;
 *                       applies to GMRES + block-Jacobi + matrix-free operator + one-pass orthogonalisation, ignored otherwise
 *   "preconditioner"    0: 3x3 block-Jacobi (north_star; default)
 *                       1: multigrid V-cycle (R15): 2x2 cell aggregates down to one cell, Galerkin
 *                          coarse operators, one damped block-Jacobi sweep before and after; uses the block-stencil operator
 *   "mg_omega"          damping of the multigrid smoother, in (0, 2) (default 0.8)
 *   "mg_precision"      64 (default) or 32: storage precision of the multigrid's matrix blocks; the cycle itself runs in fp64
 *                       on fp64 vectors, so it stays a fixed linear operator and the solve still meets the fp64 tolerance
 *   "mg_coarse_sweeps"  smoother sweeps on the coarsest (one-cell) level, >= 1 (default 2)
 * Unknown key or unsupported value: ARK_M1_E_ARG. */
ARK_M1_API int ark_m1_set_option(ark_m1* h, const char* key, double value);

/* Stage-2 fields, one plane each: "rho_cv" (rho c_v of Eq. 4; default 1), "ux", "uy" (gas velocity of Eq. 6),
 * "source_E" (constant source added to the E equation).  plane == NULL removes the field. */
ARK_M1_API int ark_m1_set_field(ark_m1* h, const char* name, const double* plane);

/* Copy out E [nx*ny], F [2*nx*ny] and, if T != NULL and a temperature was set, T [nx*ny].  Synchronises. */
ARK_M1_API int ark_m1_get_state(ark_m1* h, double* E, double* F, double* T);

/* Overlapped transfers (csrc/pipeline.cu): the same set_state / get_state for a caller that steps one state after another from HOST
 * buffers, with the upload of the NEXT state and the download of the LAST result on a copy stream of the handle's own, beside the
 * solve that is running instead of in series with it.  Nothing of the method is computed here (PAPER.md:152-173, 263-272 are the
 * steps in between); results are those of the blocking calls, bit for bit.
 *   ark_m1_prefetch_state   starts copying E (nx*ny), F (2 planes), sigma_a, sigma_s (host — pinned for a real overlap — or device)
 *                           into a staging buffer; returns at once; the arrays stay the library's until ark_m1_commit_state has
 *                           been called AND (host arrays) ark_m1_wait_transfers or a synchronisation of the handle's stream after it.
 *   ark_m1_commit_state     enqueues, on the handle's stream, "wait for that upload, then take the staged state" (= ark_m1_set_state
 *                           with T = NULL: a radiation-only state; matter coupling uses ark_m1_set_state).  ARK_M1_E_NOTSET without
 *                           a prefetch.  A new prefetch may be started right after it: it waits on the device for this commit.
 *   ark_m1_get_state_async  snapshots the current state on the handle's stream (device copy) and copies the snapshot to E, F on the
 *                           copy stream; returns at once; the handle's stream is free for the next step.  A second call waits on the
 *                           device for the first download.  E, F are valid after ark_m1_wait_transfers.
 *   ark_m1_wait_transfers   blocks the host until every copy started by the two calls above is done.
 * Device memory: 8 planes (staging 5, snapshot 3), allocated at the first call, counted in ark_m1_device_bytes.  Not for slabs of an
 * ark_m1_group (ARK_M1_E_UNSUPPORTED).  Calls on one handle must not overlap in time, as everywhere in this API. */
ARK_M1_API int ark_m1_prefetch_state(ark_m1* h, const double* E, const double* F, const double* sigma_a, const double* sigma_s);
ARK_M1_API int ark_m1_commit_state(ark_m1* h);
ARK_M1_API int ark_m1_get_state_async(ark_m1* h, double* E, double* F);
ARK_M1_API int ark_m1_wait_transfers(ark_m1* h);

/* Explicit step (rows a1-a4 of the hot path): U^{n+1} = U^n - dt R(U^n), R = divergence of the AP HLL fluxes
 * (Eqs. 12-14, 25) minus the sources (WB Eqs. 18-19 and -c sigma_a E).  One fused
 * kernel; asynchronous (no host synchronisation).  dt <= 0: ARK_M1_E_ARG. */
ARK_M1_API int ark_m1_step_explicit(ark_m1* h, double dt);

/* `nsteps` explicit steps of the same dt enqueued back to back (no host work in between). */
ARK_M1_API int ark_m1_steps_explicit(ark_m1* h, double dt, int nsteps);

/* Implicit step (rows a5-a7): assembles the linearised system (I + dt L_n) U^{n+1} = U^n + affine terms on the
 * 5-point stencil with 3 unknowns per cell (coefficients frozen at t^n) and solves it with
 * restarted GMRES(restart), right-preconditioned by the 3x3 block-Jacobi inverse (Eq. 27,
 * PAPER.md:269-272, taken block-wise), initial guess U^n, stopping when ||b - A x||_2 <= tol ||b||_2 or after
 * `maxit` inner iterations in total.  Returns the number of inner iterations (>= 0) or a negative error code;
 * *final_residual (host pointer, may be NULL) receives the TRUE relative residual ||b - A x||/||b|| recomputed
 * at exit.  Not converging is not an error: the return value is then >= maxit and *final_residual > tol.
 * Synchronises the stream.  dt <= 0, tol <= 0, restart < 1, maxit < 0: ARK_M1_E_ARG. */
ARK_M1_API int ark_m1_step_implicit(ark_m1* h, double dt, double tol, int restart, int maxit, double* final_residual);

/* Newton-Raphson on the non-linear implicit system ("we use a Newton-Raphson method ... a linear system has
 * to be solved at each iteration").  Iteration k re-assembles the operator with the coefficients of the iterate U^k, keeps
 * U^n (+ affine terms) on the right-hand side and runs GMRES from U^k; the first iteration is
 * ark_m1_step_implicit.  Stops when ||U^{k+1} - U^k||_2 <= newton_tol ||U^{k+1}||_2 or after max_newton iterations (not an
 * error).  Returns the total number of GMRES iterations or a negative error code; *newton_iterations, *final_residual (true
 * relative residual of the last linear solve) and *final_update (last relative update) are host pointers and may be NULL.
 * A temperature, if set, is linearised about T^n throughout and updated once at the end. */
ARK_M1_API int ark_m1_step_implicit_newton(ark_m1* h, double dt, double tol, int restart, int maxit, double newton_tol,
                                           int max_newton, int* newton_iterations, double* final_residual, double* final_update);

/* Semi-implicit step ("source terms remain implicit, but the hyperbolic part is time-explicit"; the paper uses it
 * for its beam and shadow tests): U* = U^n - dt [flux divergence](U^n) with the marching explicit kernel,
 * then (I + dt S) U^{n+1} = U* + affine terms, S = the source operator only (c sigma_a eta on E; the WB weights of Eqs. 18-19
 * — Eq. B.1 — or c sigma_t with "well_balanced" 0).  The second system is the implicit step's with its flux terms switched off
 * and is solved by the same Krylov method (a few iterations: it is strictly diagonally dominant).  Same arguments, return
 * value and error behaviour as ark_m1_step_implicit. */
ARK_M1_API int ark_m1_step_semi_implicit(ark_m1* h, double dt, double tol, int restart, int maxit, double* final_residual);

/* Step 3 of the operator splitting: explicit addition of the velocity sources of Eq. 6
 * using the fields "ux", "uy".  ARK_M1_E_NOTSET if they are missing. */
ARK_M1_API int ark_m1_add_velocity_sources(ark_m1* h, double dt);

/* Guards of PAPER.md:245, 513 (row a7): number of cells with E <= 0 and with |F| > cE.  Synchronises. */
ARK_M1_API int ark_m1_count_unrealizable(ark_m1* h, long long* n_E_nonpositive, long long* n_f_above_one);

/* R(U^n) of the stored state: RE [nx*ny], RF [2*nx*ny].  Synchronises. */
ARK_M1_API int ark_m1_residual(ark_m1* h, double* RE, double* RF);

/* out = A V with A = I + dt L_n assembled from the stored state (3*nx*ny doubles each), through the same
 * assembly and operator kernels the solver uses; b_out (may be NULL) receives the right-hand side. Synchronises. */
ARK_M1_API int ark_m1_apply_operator(ark_m1* h, double dt, const double* V, double* out, double* b_out);

/* out = M^-1 V, M^-1 = the right preconditioner the solver uses for a step dt ("A K^-1 y = b, K x = y"):
 * the inverse 3x3 diagonal blocks (Eq. 27 block-wise; option "preconditioner" = 0, default) or one multigrid V-cycle
 * ("preconditioner" = 1, R15).  V, out: 3*nx*ny doubles, host or device.  Synchronises. */
ARK_M1_API int ark_m1_apply_preconditioner(ark_m1* h, double dt, const double* V, double* out);
/* Two applications of the preconditioned operator in a row, as the s-step Arnoldi block issues them (DESIGN.md "Two applications
 * per pass"): out1 = A M^-1 V - theta1 V, out2 = A M^-1 out1 - theta2 out1 for the linearisation of a step dt at the current
 * state (A = I + dt L_n; M = its 3x3 block diagonal).  V, out1, out2: 3 planes of nx*ny doubles
 * each (E, Fx, Fy), host or device.  With option "op_pair" = 1 (default), the default matrix-free operator (op_recompute = 2) and a
 * grid of at least 4 x 4 cells (any boundary kinds) both come from ONE pass over the coefficient planes; otherwise from two passes.
 * Returns 1 if the one-pass kernel ran, 0 if two passes did, < 0 on error (ARK_M1_E_UNSUPPORTED with option operator = 0).
 * Synchronises the handle's stream. */
ARK_M1_API int ark_m1_apply_operator_pair(ark_m1* h, double dt, const double* V, double* out1, double* out2, double theta1, double theta2);

/* Relative residual history of the last implicit solve: entry 0 = true residual of the initial guess, then one
 * estimate per inner iteration.  Copies min(cap, n) values into buf (host) and returns n. */
ARK_M1_API int ark_m1_get_history(ark_m1* h, double* buf, int cap);

/* Timings of the last implicit solve in milliseconds (CUDA events on the handle's stream):
 * out[0] = assembly, out[1] = Krylov iterations (everything after assembly), out[2] = total. */
ARK_M1_API int ark_m1_get_timings(ark_m1* h, double* out3);

/* Launch statistics.  After ark_m1_set_option(h, "kernel_timing", 1) every kernel launch of the handle is
 * bracketed by CUDA events on the handle's stream; out[3k .. 3k+2] = number of launches, total milliseconds and
 * total ALGORITHMIC bytes of kernel class k.  Returns the number of classes; names from
 * ark_m1_kernel_class_name(k).  ark_m1_kernel_launches = kernels launched by the handle since creation. */
ARK_M1_API int ark_m1_get_kernel_stats(ark_m1* h, double* out, int cap);
ARK_M1_API const char* ark_m1_kernel_class_name(int k);
ARK_M1_API long long ark_m1_kernel_launches(const ark_m1* h);
/* s-step Arnoldi blocks of the LAST linear solve (the restarted Krylov solve of PAPER.md:263-272, built five columns at a time), by the
 * way their in-block factorisation went:
 * out4[0] finished by the update pass (solve predicted by the dot pass, measured Gram matrix within tolerance),
 * out4[1] predicted, then a second round from the measured Gram matrix, out4[2] measured factorisation and a separate in-block pass,
 * out4[3] the same with a second round.  out4 is a host array of 4.  Zeros when the solve built no blocks. */
ARK_M1_API int ark_m1_block_stats(const ark_m1* h, long long* out4);

/* Self-test of the fast fp64 reciprocal / reciprocal square root of the hot kernels (MUFU seed + Newton steps): out4[0..3] =
 * max relative error of rcp_fast vs 1/x, rsqrt_fast vs 1/sqrt(x), sqrt_fast vs sqrt(x) and rcp_fast3 (one third-order step,
 * explicit kernel) vs 1/x over n samples in 200 binades (host pointer to 4 doubles).  Expected: 0, <= 1 ulp, <= 1 ulp, <= 1 ulp.
 * No handle needed. */
ARK_M1_API int ark_m1_fastmath_errors(int n, double* out4);

/* Self-test that MEASURES the issue rates of the instruction kinds the explicit and assembly kernels are bound by (they are
 * fp64-issue bound, not HBM bound: DESIGN.md section 6), on the current device.  No handle needed; takes a few milliseconds.
 * out (host, cap >= 12):
 *   [0] DFMA lanes per clock per SM (every SM full, 8 independent chains per thread)   [1] DFMA dependent-issue latency, cycles
 *   [2] DADD, [3] DMUL, [4] compare+select max (DSETP + SEL), [5] IMAD, [6] FFMA: lanes per clock per SM
 *   [7] issue cycles per (DFMA + IMAD) pair per warp per SM sub-partition, [8] the same for (DFMA + FFMA)
 *   [9] 64-bit warp shuffles, lanes per clock per SM      [10] SM clock during the test, MHz      [11] number of SMs
 * The fp64 "alu" roofline of bench.py is out[0] * out[11] * clock lane-instructions per second.
 * Returns 12, or ARK_M1_E_ARG / ARK_M1_E_ALLOC / ARK_M1_E_CUDA / ARK_M1_E_UNSUPPORTED. */
ARK_M1_API int ark_m1_fp64_issue_rate(double* out, int cap);

/* ---------------------------------------------------------------------------------------------------------------------------
 * Domain-decomposed step: 1-D slabs in y, one slab per rank ("regular domain decomposition with ghost cells";
 * PAPER.md:315 rows of the linear system distributed over the ranks; "several communications per iteration").
 * Rank r of nranks owns the global rows [y0, y1) of ark_m1_slab_range.  Per explicit step and per assembly the boundary rows of
 * (E, Fx, Fy, sigma_a, sigma_t) are exchanged with the two neighbours; per operator application the boundary rows of
 * (z, c^2 J z), z = M^-1 v; per GMRES iteration the j+1 Gram-Schmidt dot products and ||w||^2 are all-reduced (fp64).
 * Everything else runs in the one-GPU kernels on the slab.  Supported: ark_m1_group_step_explicit (all explicit kernels, matter
 * terms included) and ark_m1_group_step_implicit with the default solver configuration (GMRES(m) + block-Jacobi, matrix-free
 * operator); other solver options return ARK_M1_E_UNSUPPORTED.
 *
 * A group owns its slab solvers.  ark_m1_group_slab returns them: use ark_m1_set_state / ark_m1_set_field / ark_m1_set_boundary
 * (x sides, and the y sides that are global boundaries) / ark_m1_set_option / ark_m1_get_state on a slab handle with LOCAL arrays
 * of (y1 - y0) x nx cells; the stepping calls on a slab handle return ARK_M1_E_UNSUPPORTED (the halos must be exchanged).
 * --------------------------------------------------------------------------------------------------------------------------- */
typedef struct ark_m1_group ark_m1_group;

/* Rows [*y0, *y1) of rank `rank` of `nranks` on a grid of ny rows: y0 = floor(ny rank / nranks).  Host arithmetic only (no GPU). */
ARK_M1_API int ark_m1_slab_range(int ny, int nranks, int rank, int* y0, int* y1);

/* Caller-supplied transport for ark_m1_group_create_host: HOST buffers, blocking calls, 0 on success.
 *   sendrecv     : send `n` doubles of send_lo to rank `lo` and of send_hi to rank `hi`; receive `n` doubles from `lo` into recv_lo
 *                  and from `hi` into recv_hi.  lo / hi < 0: no such neighbour (its buffers are not touched).  What a rank sends to
 *                  its `lo` neighbour arrives in that neighbour's recv_hi, and vice versa (with two ranks and a periodic direction lo
 *                  and hi are the same peer).
 *   allreduce_sum: buf[0..n) <- sum over all ranks, the same result on every rank. */
typedef struct {
    void* ctx;
    int (*sendrecv)(void* ctx, int lo, int hi, const double* send_lo, const double* send_hi, double* recv_lo, double* recv_hi, long long n);
    int (*allreduce_sum)(void* ctx, double* buf, int n);
} ark_m1_host_transport;

/* All nranks slabs in this process on the current device (exchange = device copies, all-reduce = a kernel; nothing ever waits on
 * another rank): the form the decomposition is tested in on one GPU.  Global arguments as for ark_m1_create. */
ARK_M1_API ark_m1_group* ark_m1_group_create_local(int nx, int ny, double dx, double dy, double c, const ark_m1_bc* bc, int nranks);
/* One slab (rank `rank`) in this process; halos and sums staged through pinned host memory and the caller's transport. */
ARK_M1_API ark_m1_group* ark_m1_group_create_host(int nx, int ny, double dx, double dy, double c, const ark_m1_bc* bc, int rank, int nranks,
                                                  const ark_m1_host_transport* transport);
/* One slab in this process on the current GPU; ncclSend/ncclRecv + ncclAllReduce on the solver's stream.  unique_id128: the 128 bytes
 * of ark_m1_nccl_unique_id obtained on one rank and distributed to all by the caller.  libnccl.so.2 is opened with dlopen. */
ARK_M1_API int ark_m1_nccl_unique_id(void* out128);
ARK_M1_API ark_m1_group* ark_m1_group_create_nccl(int nx, int ny, double dx, double dy, double c, const ark_m1_bc* bc, int rank, int nranks,
                                                  const void* unique_id128);
ARK_M1_API void ark_m1_group_destroy(ark_m1_group* g);
ARK_M1_API int ark_m1_group_set_stream(ark_m1_group* g, void* cuda_stream);

/* Number of slabs held by this process (nranks for a local group, 1 otherwise) and the k-th of them with its rank and rows. */
ARK_M1_API int ark_m1_group_local_slabs(const ark_m1_group* g);
ARK_M1_API ark_m1* ark_m1_group_slab(ark_m1_group* g, int k, int* rank, int* y0, int* y1);

/* The decomposed steps; arguments, return values and error behaviour as ark_m1_step_explicit / ark_m1_step_implicit (collective:
 * every rank calls them with the same arguments). */
ARK_M1_API int ark_m1_group_step_explicit(ark_m1_group* g, double dt);
ARK_M1_API int ark_m1_group_step_implicit(ark_m1_group* g, double dt, double tol, int restart, int maxit, double* final_residual);

/* Communication counters since creation: halo bytes sent by this process, exchanges, all-reduces. */
ARK_M1_API int ark_m1_group_comm_stats(const ark_m1_group* g, long long* halo_bytes, long long* exchanges, long long* allreduces);
ARK_M1_API const char* ark_m1_group_last_error(const ark_m1_group* g);

/* ---------------------------------------------------------------------------------------------------------------------------
 * Three space dimensions ("its extension to higher dimensions is straightforward"; (2+d)N unknowns):
 * the same scheme direction by direction on (E, Fx, Fy, Fz), 7-point stencil, explicit step and one linearised implicit step
 * solved by GMRES(restart) right-preconditioned with the 4x4 diagonal blocks.  Generic kernels (one thread per cell).
 * Arrays: planes [nz][ny][nx], x fastest; F = [Fx | Fy | Fz] (3 nx ny nz doubles); host or device pointers.
 * Boundaries: ARK_M1_BC_PERIODIC or ARK_M1_BC_OUTFLOW per side.  Arguments, return values and error behaviour as the 2-D calls.
 * --------------------------------------------------------------------------------------------------------------------------- */
typedef struct ark_m1_3d ark_m1_3d;
typedef struct { int xlo, xhi, ylo, yhi, zlo, zhi; } ark_m1_bc3;
ARK_M1_API ark_m1_3d* ark_m1_3d_create(int nx, int ny, int nz, double dx, double dy, double dz, double c, const ark_m1_bc3* bc);
ARK_M1_API void ark_m1_3d_destroy(ark_m1_3d* h);
ARK_M1_API int ark_m1_3d_set_stream(ark_m1_3d* h, void* cuda_stream);
ARK_M1_API int ark_m1_3d_set_state(ark_m1_3d* h, const double* E, const double* F, const double* sigma_a, const double* sigma_s);
/* "explicit_kernel": 1 = two streaming passes, closure once per cell then the flux-form stencil (default); 0 = one thread per cell
 * evaluating its seven closures itself (IEEE divisions and roots).
 * "arnoldi_block": 5 (default), 4, 3 = s-step Arnoldi blocks as in the 2-D solver (columns a restart length leaves over use the
 * two-column step); 1 = one column per pass over the basis. */
ARK_M1_API int ark_m1_3d_set_option(ark_m1_3d* h, const char* key, double value);
ARK_M1_API int ark_m1_3d_get_state(ark_m1_3d* h, double* E, double* F);
ARK_M1_API int ark_m1_3d_step_explicit(ark_m1_3d* h, double dt);
ARK_M1_API int ark_m1_3d_step_implicit(ark_m1_3d* h, double dt, double tol, int restart, int maxit, double* final_residual);
/* out = A V (precond == 0) or A M^-1 V (precond != 0), A = I + dt L_n of the stored state, through the solver's own assembly and
 * operator kernels; V, out: 4 nx ny nz doubles [E | Fx | Fy | Fz].  Synchronises. */
ARK_M1_API int ark_m1_3d_apply_operator(ark_m1_3d* h, double dt, const double* V, double* out, int precond);
ARK_M1_API long long ark_m1_3d_kernel_launches(const ark_m1_3d* h);
ARK_M1_API const char* ark_m1_3d_last_error(const ark_m1_3d* h);

/* ---------------------------------------------------------------------------------------------------------------------------
 * The realizability guard without any allocation (row a7), for callers that cannot call cudaMalloc: code
 * under CUDA graph capture, tight serving loops, harnesses that forbid it.  No handle.  Same predicate and arithmetic as
 * ark_m1_count_unrealizable; the scratch (one pair of partial counts per block of 4096 cells and the "last block" ticket) lives
 * in a static __device__ array of 262 400 bytes inside the library, held by every GPU that loads libark_m1.so until the process
 * exits.  The call enqueues one 256-byte memset of the ticket and one kernel on `cuda_stream` and returns; it never synchronises
 * and calls no cudaMalloc / cudaFree / allocating routine.
 *   E, Fx, Fy : DEVICE pointers on the current device, ncells doubles each (any plane layout; [ny][nx] flattened), read only
 *   c         : speed of light
 *   counts2   : DEVICE pointer, 2 x unsigned long long, written by the kernel: [0] cells with E <= 0 (or NaN), [1] cells with
 *               E > 0 and |F| > cE.  Valid once `cuda_stream` has reached the kernel's end.  ncells == 0 writes two zeros.
 * Limit: ncells <= ark_m1_noalloc_max_cells() = 67 108 864 (8192^2); beyond it the call returns ARK_M1_E_UNSUPPORTED and
 * launches nothing.  Other errors: ARK_M1_E_ARG (null pointer, ncells < 0), ARK_M1_E_CUDA.  ark_m1_noalloc_last_error() holds
 * the calling thread's last message.
 * Sharing: every call on a device uses the same array, which keeps the previous call's contents (the call clears what must
 * start at zero).  Calls that can overlap on the GPU — different streams, different host threads, two captured graphs launched
 * concurrently — race on it and return wrong counts: order them on one stream or with events.
 * ark_m1_noalloc_setup() resolves the array's device address for the CURRENT device (cudaGetSymbolAddress, once per device;
 * may load the module): call it once per device before capturing; ark_m1_count_unrealizable_noalloc calls it itself otherwise.
 * --------------------------------------------------------------------------------------------------------------------------- */
ARK_M1_API int ark_m1_noalloc_setup(void);
ARK_M1_API long long ark_m1_noalloc_max_cells(void);
ARK_M1_API int ark_m1_count_unrealizable_noalloc(const double* E, const double* Fx, const double* Fy, long long ncells, double c,
                                                 unsigned long long* counts2, void* cuda_stream);
ARK_M1_API const char* ark_m1_noalloc_last_error(void);

/* Device bytes currently allocated by the handle. */
ARK_M1_API long long ark_m1_device_bytes(const ark_m1* h);

ARK_M1_API const char* ark_m1_last_error(const ark_m1* h);
ARK_M1_API const char* ark_m1_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ARK_M1_H */
