/* gmmnlse.h -- C ABI of the B200-native GMMNLSE / MPA hot path.
 *
 * Method: Wright et al., "Multimode Nonlinear Fiber Optics: Massively Parallel
 * Numerical Solver, Tutorial and Outlook", arXiv 1708.05324.  Citations are
 * PAPER.md line numbers.
 *
 *   Eq. 1   the GMMNLSE right-hand side
 *   Eq. 2   S^K = S^R = S, real, from real scalar mode fields
 *   Eq. 11  A_p(z,w) = psi_p(z,w) exp[D_w (z - z0)]
 *   Eq. 12  integral form; PAPER.md:214-218 the M-plane iteration
 *
 * Conventions (reading S1): F{f}_k = sum_n f_n exp(+2 pi i k n/N),
 * w_k = 2 pi k'/(N dt) (k' = k for k < N/2, else k - N), d/dt <-> -i w,
 * D_w^(p) = i[beta0 + beta1 w + sum_{k>=2} beta_k w^k/k!].
 *
 * All work runs in hand-written sm_100a kernels; there is no CPU fallback.
 * Every call returns GMMNLSE_OK (0) on success, a negative code on failure and
 * (propagate only) the positive GMMNLSE_WARN_NOCONV when some large step hit
 * max_iter.  No exception crosses this boundary; on GMMNLSE_EINVAL no output is
 * written.  A plan is not thread-safe; use one plan per host thread.
 */
#ifndef GMMNLSE_H_
#define GMMNLSE_H_

#ifdef __cplusplus
extern "C" {
#endif

#define GMMNLSE_OK            0
#define GMMNLSE_WARN_NOCONV   1   /* >=1 large step stopped at max_iter; last iterate used   */
#define GMMNLSE_EINVAL       -1   /* bad argument (see each call)                            */
#define GMMNLSE_ENOMEM       -2   /* host or device allocation failed                        */
#define GMMNLSE_ECUDA        -3   /* a CUDA call failed; see gmmnlse_last_cuda_error()        */
#define GMMNLSE_EUNSUPPORTED -4   /* legal request outside what the kernels cover             */

typedef struct gmmnlse_plan gmmnlse_plan;   /* opaque; owns every device buffer it allocates */

typedef struct {                /* pass NULL for defaults                                        */
  int    precision;             /* 0 = complex64 (default), 1 = complex128                        */
  int    shock;                 /* 1 (default): factor (1 + w/w0) of Eq. 12 on; 0: off            */
  double tol;                   /* MPA convergence threshold, default 1e-6         */
  int    max_iter;              /* cap on iterations per large step; <=0 -> 2*M + 4               */
  int    fixed_iter;            /* >0: run exactly this many iterations per large step (parity)   */
  int    contraction;           /* a6 kernel: 0 = auto (complex64, N % 128 == 0 and Q = P(P+1)/2 >= 64: 7; else 1),
                                   1 = CUDA-core fp32/fp64 GEMM;
                                   3 = tcgen05 3xTF32 GEMM (kind::tf32 on hi/lo splits, both operands in shared memory);
                                   7 = tcgen05 kind::f16 GEMM on fp16 hi/lo splits of both operands (22 mantissa
                                   bits, as 3xTF32, at twice its MMA rate): the pair kernels write V scaled by a
                                   power of two into fp16 range as two fp16 arrays, S is split per row at plan
                                   time, the scales are undone exactly in the epilogue;
                                   6 = exact low-rank form on the 3xTF32 kernel,
                                   8 = the same on the kind::f16 kernel: S_(pl),(mn) = sum_k L_(pl),k L_(mn),k
                                   by pivoted Cholesky at plan time (Eq. 2 makes S a Gram matrix; rank 153 of
                                   1035 for 45 Hermite-Gauss modes), two GEMMs Q x R and R x Q instead of Q x Q;
                                   EUNSUPPORTED if S is not positive semi-definite;
                                   9 = block-sparse form of the dense product on the kind::f16 kernel: the packed
                                   pairs fall into classes that S never couples (the parities of F_p F_l in x and
                                   y for Hermite-Gauss modes: Eq. 2's integrand is odd otherwise), found at plan
                                   time as the connected components of |S2| > 1e-13 max|S2|; operands are stored
                                   in class order and every output tile multiplies only its own class's blocks
                                   (about 1/4 of the multiply-adds for a GRIN fibre).  Same result as 7 up to the
                                   dropped entries; EUNSUPPORTED if there is one class only or on a general plan.
                                   6, 8, 9 are never chosen by auto: BASELINE.json names the dense contraction.
                                   3-9 need complex64 and N % 128 == 0, else EUNSUPPORTED.  Other values: EINVAL */
  int    raman;                 /* a5 kernel: 0 = auto, 1 = FFT . h~_R . IFFT on the pair streams (any h_R),
                                   2 = one-pole recurrence along t, exact when the samples are a damped
                                   oscillation h_R[j] = Im(c zeta^j) (the tau1/tau2 form); auto picks 2 when
                                   all N samples fit that form to 1e-10 of the peak, else 1; 2 on a response
                                   that does not fit is EUNSUPPORTED                                */
  int    graph;                 /* MPA iteration loop: 0 (default) = on the device -- every full
                                   large step is one CUDA graph (iteration 0, a WHILE node whose body is one
                                   further iteration, a11); the convergence test err < tol and the max_iter cap
                                   are evaluated by a kernel that sets the node's condition, and the host reads
                                   the counters back once per gmmnlse_propagate call.  1 = host loop: one 8-byte
                                   D2H and a stream synchronise per iteration.  Same kernels, same arithmetic,
                                   same iteration counts.  The first large step of a plan, a ragged last step
                                   ((L/dz) mod M planes) and calls under gmmnlse_profile_enable use the host
                                   loop in either case                                               */
  int    stop_rule;             /* when an MPA large step counts as converged ("once the accuracy reaches a
                                   given threshold"): 0 (default, reading S12) = err_n < tol, err_n the
                                   relative change of the planes in iteration n; 1 (reading S25) = also when the
                                   a-posteriori bound on the iterate's distance to the fixed point,
                                   err_n rho / (1 - rho) with rho the larger of the last two ratios err_n / err_{n-1}
                                   (n >= 3), is below tol.  Per large step the result differs by less than tol and
                                   takes one iteration less wherever the last one only confirmed convergence; the
                                   steps then end at an error near tol instead of ~10x below it, and these residuals
                                   add up over the large steps (measured: photon number +1.7e-7 per large step at
                                   tol = 1e-6) -- lower tol for long runs with tight invariants.  Other values: EINVAL */
  int    async_call;            /* 0 (default): gmmnlse_propagate returns after one synchronise that follows its last
                                   kernel (A_out complete, counters current, WARN_NOCONV reported by the return code).
                                   1: with the loop on the device (options.graph = 0) the call returns as soon as its
                                   work is enqueued -- A_out is complete once the stream is synchronised, the return
                                   code is OK, and the loop counters (iterations, not_converged, last_err) are taken
                                   in lazily by the next gmmnlse_get_stats / gmmnlse_launch_count / propagate call,
                                   which waits for the stream if it has to.  Large steps that run on the host loop
                                   (a plan's first one, a ragged last one, profiling) still synchronise per
                                   iteration; gmmnlse_propagate_host always synchronises.  Other values: EINVAL   */
} gmmnlse_options;

/* Build a plan: precompute D_w^(p), the rotation tables exp(+-D_w j dz) (j = 0..M) in
 * fp64, K(w) = i n2 w0/c (1 + w/w0), the blended Raman transfer function
 * (1 - fR) + fR dt F{h_R}, and the pair-packed coupling matrix.
 *
 *   P, N, M   modes, time samples (power of two, 16 <= N <= 16384; complex128: N <= 8192),
 *             small steps per large step (>= 1)
 *   dt, dz    time-grid spacing [s]; small step [m]
 *   beta      HOST [P][n_beta], beta[p*n_beta + k] = beta_k^(p) in s^k/m
 *             (k = 0: delta-beta0 [1/m], k = 1: delta-beta1 [s/m])  (Eq. 1 terms 1-3)
 *   S         HOST [P][P][P][P], index ((p*P + l)*P + m)*P + n, in 1/m^2 (Eq. 2).  Must be
 *             symmetric under m<->n and p<->l (true for Eq. 2); otherwise EUNSUPPORTED.
 *   f_R, h_R  Raman fraction; HOST [N] samples h_R(j dt) in 1/s (NULL iff f_R == 0)
 *   omega0    carrier [rad/s];  n2 [m^2/W]
 * Host arrays are copied; the caller keeps ownership.  The plan lives on the CUDA device that is
 * current at creation; every later call runs there whatever the caller's current device.
 * EINVAL: sizes < 1, N not a power of two, pi/dt >= omega0 with shock on, NULL pointers,
 * non-finite beta/S/h_R, f_R outside [0, 1].                                              */
int gmmnlse_plan_create(gmmnlse_plan **out, int P, int N, int M, double dt, double dz,
                        const double *beta, int n_beta, const double *S,
                        double f_R, const double *h_R, double omega0, double n2,
                        const gmmnlse_options *opt);

/* Plan for the GENERAL form of Eq. 1: separate Kerr and Raman tensors,
 *   N_p = sum_lmn A_l [(1-fR) S^K_plmn A_m A_n* + fR S^R_plmn (h_R (*) A_m A_n*)],
 * real or complex, with NO index symmetry assumed.  Two polarisations per spatial mode are 2P fields with the
 * corresponding (2P)^4 tensors.  S_K, S_R: HOST [P][P][P][P] (index as S above), doubles; if tensors_complex != 0
 * each entry is (re, im) interleaved.  Everything else as gmmnlse_plan_create; all other calls work on the plan
 * unchanged.  The contraction runs on 2 ceil(P^2/2) x 2 real pair streams (Re and Im of A_m A_n*, Kerr- and
 * Raman-weighted) instead of the P(P+1)/2 packed ones: about 8x the work of the scalar-mode path at equal P.   */
int gmmnlse_plan_create_general(gmmnlse_plan **out, int P, int N, int M, double dt, double dz,
                                const double *beta, int n_beta, const double *S_K, const double *S_R,
                                int tensors_complex, double f_R, const double *h_R, double omega0, double n2,
                                const gmmnlse_options *opt);

/* Integrate Eq. 1 from z0 to z0 + L with the MPA.
 *   A_in, A_out  DEVICE [P][N] interleaved (re,im), float2 or double2 per precision, time
 *                domain, sqrt(W); A_out may alias A_in; never freed by the library.
 *   L            [m], an integer multiple of dz (1e-9 relative) else EINVAL; the last large
 *                step uses (L/dz) mod M planes.
 *   stream       cudaStream_t as void*; applies to THIS call only (NULL = the plan's stream, see
 *                gmmnlse_set_stream).  Work is enqueued on it and the call returns after one
 *                synchronise that follows the last kernel: A_out is complete on return and the
 *                counters of gmmnlse_get_stats are current (the return code WARN_NOCONV needs
 *                them).  Device loop (options.graph = 0): that is the only synchronise of the
 *                call; host loop: one 8-byte D2H + synchronise per iteration as well.  `stream`
 *                must not be capturing.                                                     */
int gmmnlse_propagate(gmmnlse_plan *plan, const void *A_in, double L, void *A_out, void *stream);

/* Same as gmmnlse_propagate but A_in / A_out are HOST [P][N] buffers of the plan's
 * precision: H2D copy, propagate, D2H copy on the plan's stream, one synchronise; A_out is
 * complete on return.  Page-locked buffers (cudaMallocHost / cudaHostRegister) are copied
 * from and to directly; pageable ones are staged through plan-owned pinned memory; device or
 * managed pointers are EINVAL (use gmmnlse_propagate).  This is the end-to-end entry
 * bench.py times (with page-locked buffers).                                               */
int gmmnlse_propagate_host(gmmnlse_plan *plan, const void *A_in_host, double L, void *A_out_host);

/* Serial comparison integrator (the role of the split-step code the paper times the
 * MPA against): fixed-step fourth-order Runge-Kutta in the interaction picture
 * (RK4IP) with step dz, four nonlinear-operator evaluations per step through the same a3-a8 kernels, one
 * plane per launch.  Arguments, layout and errors as gmmnlse_propagate; fully asynchronous (no read-back).  */
int gmmnlse_propagate_rk4ip(gmmnlse_plan *plan, const void *A_in, double L, void *A_out, void *stream);

/* Other effects within the GMMNLSE (section F), both integrators:
 *   set_gain:     small-signal FIELD gain g_p A_p; g: HOST [P] in 1/m (negative = loss), NULL or all
 *                 zero = none.  Linear and diagonal, so it joins D_w as its real part: the rotation tables
 *                 exp(+-D_w j dz) get the factors exp(+-g_p j dz).  Frequency-independent gain only.
 *   set_gain_saturation: first-order saturation of that gain (the Taylor expansion of
 *                 g(I) = g0 / [1 + int dt I / I_sat] projected on the modes), the additional term
 *                   - g_sat sum_lmn S_plmn A_l(t) int dtau A_m(tau) A_n*(tau),    g_sat = g0 / I_sat in m/J
 *                 (the paper prints the term without its gain prefactor: DESIGN.md reading S22); the time integral is
 *                 dt sum_t over the window.  0 = off.  Scalar-mode plans only (EUNSUPPORTED on a general plan).
 *   set_coupling: linear mode coupling C_p = i sum_n Q_np A_n (Eq. 13 for Q_np); Q: HOST [P][P]
 *                 (re, im) interleaved, entry (n P + p) = Q_np in 1/m, NULL or all zero = none.  Constant over
 *                 frequency.  Integrated with the nonlinear term (same trapezoid / RK4 stages).
 *   set_coupling_profile: z-dependence of the coupling, Q(z) = f(z) Q: the separable index perturbation
 *                 eps(x, y) f(z) of PAPER.md:277 (a grating: f periodic; disorder: f a stochastic function).  f: HOST
 *                 [n] samples f(k dz / 2), k = 0..n-1, measured from the START of each propagate call (the RK4IP
 *                 stages sit on half steps; the MPA planes use the even samples); a call over L needs
 *                 n >= 2 L / dz + 1, else EINVAL.  NULL = constant coupling (f = 1).
 * gmmnlse_nonlinear_op includes none of these.  All four synchronise the plan's stream, copy their argument, and
 * return EINVAL on non-finite input.                                                                              */
int gmmnlse_set_gain(gmmnlse_plan *plan, const double *g);
int gmmnlse_set_coupling(gmmnlse_plan *plan, const double *Q);
int gmmnlse_set_coupling_profile(gmmnlse_plan *plan, const double *f, int n);
int gmmnlse_set_gain_saturation(gmmnlse_plan *plan, double g_sat);

/* Plane-axis sharding of one MPA large step over several GPUs (the M planes are
 * the parallel axis).  Every shard holds a plan of the SAME arguments on its own device and owns the planes
 * j_lo+1 .. j_hi of the current large step's Mc planes (shard 0 also plane 0); the collectives between the calls are
 * the caller's (paper_1708_05324_b200/sharded.py drives them over NCCL), all pointers are DEVICE pointers:
 *   shard_begin(A_in)                  psi_0 = F{A_in}, on every shard                                        (a1)
 *   repeat
 *     shard_iterate(j_lo, j_hi, Mc, first, block_sum)
 *                                      a3-a8 on the shard's planes; block_sum [P][N] <- sum_j w_j G_j over them,
 *                                      w = 1/2 on planes 0 and Mc, else 1 (trapezoid rule).
 *                                      first != 0: the first iterate psi_j = psi_0 (and shard 0 forms G_0)
 *     -- all-gather of the block sums -> all_sums [n_shards][P][N], shard order --
 *     shard_update(..., all_sums, shard, n_shards, &err_local)
 *                                      a9 on the shard's planes from the exclusive prefix of the block sums;
 *                                      err_local = max over ITS planes of |psi_new - psi_old| / |psi_new| (a10);
 *                                      synchronises the stream (8-byte read-back)
 *     -- max all-reduce of err_local; stop when < tol or at max_iter --
 *   shard_advance(Mc, all_sums, n_shards)   psi_0 <- (psi_0 + dz sum_g block_g) exp(D Mc dz) on every shard   (a11)
 *   shard_end(A_out)                   A_out = F^-1{psi_0}
 * With n_shards = 1 (j_lo = 0, j_hi = Mc) the sequence is the host loop of gmmnlse_propagate.  EINVAL on plane
 * ranges outside 0 <= j_lo < j_hi <= Mc <= M.  The counters of gmmnlse_get_stats count this shard's calls.      */
int gmmnlse_shard_begin(gmmnlse_plan *plan, const void *A_in);
int gmmnlse_shard_iterate(gmmnlse_plan *plan, int j_lo, int j_hi, int Mc, int first, void *block_sum);
int gmmnlse_shard_update(gmmnlse_plan *plan, int j_lo, int j_hi, int Mc, int first, const void *all_sums, int shard,
                         int n_shards, double *err_local);
int gmmnlse_shard_advance(gmmnlse_plan *plan, int Mc, const void *all_sums, int n_shards);
int gmmnlse_shard_end(gmmnlse_plan *plan, void *A_out);

/* One evaluation of the last term of Eq. 1:
 *   dA_p(t) = i n2 w0/c (1 + i/w0 d_t) sum_lmn S_plmn A_l [(1-fR) A_m A_n* + fR (h_R (*) A_m A_n*)]
 * A, dA: DEVICE [P][N] as above (dA must not alias A); enqueued on the plan's stream.      */
int gmmnlse_nonlinear_op(gmmnlse_plan *plan, const void *A, void *dA);

/* Bind the plan to a stream: every later call that is given no stream of its own (NULL, or calls without a
 * stream argument: nonlinear_op, propagate_host, the debug_* stages) enqueues there.  Default: the NULL stream. */
int gmmnlse_set_stream(gmmnlse_plan *plan, void *stream);

/* Counters accumulated since plan creation (any pointer may be NULL).                      */
int gmmnlse_get_stats(const gmmnlse_plan *plan, long long *large_steps, long long *iterations,
                      double *last_err, long long *not_converged);

/* Kernel launches issued by this plan since creation (bench.py's "gpu_launches").          */
long long gmmnlse_launch_count(const gmmnlse_plan *plan);

/* Per-kernel-class device timing with CUDA events recorded on the plan's stream around every
 * launch (bench.py's roofline numbers).  enable(on=1) clears the accumulators; get() synchronises
 * the stream and returns the summed duration [ms] and launch count of one kernel class.        */
#define GMMNLSE_KIND_FFT_TO_TIME 0   /* a3 (+ final inverse transform): psi_j E+_j -> A_j(t)      */
#define GMMNLSE_KIND_PAIR_CONV   1   /* a4 + a5: pair products, Raman FFT.h.IFFT, blend            */
#define GMMNLSE_KIND_CONTRACT    2   /* a6: S contraction                                          */
#define GMMNLSE_KIND_MODE_REDUCE 3   /* a7: sum_l U_pl A_l                                         */
#define GMMNLSE_KIND_FFT_TO_FREQ 4   /* a1, a8: F{.} K(w) E-_j                                      */
#define GMMNLSE_KIND_SCAN        5   /* a9 + a10: trapezoid scan over planes + error norms        */
#define GMMNLSE_KIND_ADVANCE     6   /* a11: plane shift                                           */
#define GMMNLSE_KIND_MISC        7   /* conversions, error finalisation                            */
#define GMMNLSE_KIND_COUNT       8
int gmmnlse_profile_enable(gmmnlse_plan *plan, int on);
int gmmnlse_profile_get(gmmnlse_plan *plan, int kind, double *total_ms, long long *launches);

/* Parity hook: copy the interaction-picture planes psi_j (j = 0..M) of the most recent large
 * step to HOST out[(M+1)][P][N] (precision of the plan).  Synchronises the stream.         */
int gmmnlse_debug_get_planes(gmmnlse_plan *plan, void *out_host);

/* Stage-level entry points used by the unit tests and micro-benchmarks (DEVICE pointers).
 *   fft:   rows x N transform of the plan's precision; dir = +1 to-frequency (un-normalised,
 *          exp(+i..)), -1 to-time (exp(-i..), scaled by 1/N).  out may alias in.
 *   pairs: V[q][t] = (1-fR) Re T_mn + fR (h_R (*) Re T_mn), q = packed pair index of m <= n,
 *          for n_planes planes of A [plane][P][N]  ->  V [plane][Q][N] (real).             */
int gmmnlse_debug_fft(gmmnlse_plan *plan, const void *in, void *out, int rows, int dir);
int gmmnlse_debug_pairs(gmmnlse_plan *plan, const void *A, void *V, int n_planes);
/*   contract: U[plane][r][t] = sum_q S2[r][q] V[plane][q][t] over packed pairs r = (p<=l), q = (m<=n),
 *          S2 = S_plmn with the m<n columns doubled (Eq. 1's sum over m,n); V, U DEVICE
 *          [n_planes][Q][N] real of the plan's precision, U must not alias V.
 *   contraction_kind: which a6 kernel the plan selected (the values of options.contraction): 1 CUDA cores,
 *          3 tcgen05 3xTF32, 6 low-rank pair of 3xTF32 GEMMs, 7 tcgen05 kind::f16 on fp16 hi/lo splits,
 *          8 low-rank pair of kind::f16 GEMMs, 9 block-sparse kind::f16.  With 7 and 8 debug_pairs still writes fp32 V, and
 *          debug_contract splits the caller's fp32 V into fp16 pairs first (scaled by its own max |V|).                                                            */
int gmmnlse_debug_contract(gmmnlse_plan *plan, const void *V, void *U, int n_planes);
int gmmnlse_contraction_kind(const gmmnlse_plan *plan);
/*   lowrank_rank: rank R of the factorisation when contraction_kind is 6 or 8, else 0.            */
int gmmnlse_lowrank_rank(const gmmnlse_plan *plan);
/*   sparse_info: contraction_kind 9: number of uncoupled classes of packed pairs and the fraction of the dense
 *          multiply-adds the block-sparse form executes (padding included); otherwise 0 and 1.  Pointers may be NULL. */
int gmmnlse_sparse_info(const gmmnlse_plan *plan, int *classes, double *work_fraction);
/*   loop_kind: how the MPA iteration loop of the last gmmnlse_propagate ran: 1 = on the device (CUDA-graph
 *          WHILE node, options.graph = 0), 0 = host loop only so far, -1 = the graph could not be built on this
 *          driver and the plan fell back to the host loop (gmmnlse_last_cuda_error() says why).          */
int gmmnlse_loop_kind(const gmmnlse_plan *plan);
/*   raman_kind: which a5 kernel the plan selected: 0 none (f_R = 0), 1 FFT, 2 recursive.          */
int gmmnlse_raman_kind(const gmmnlse_plan *plan);
/*   set_tc_chunk: k-blocks (16 packed pairs each in the 3xTF32 forms, 32 in the kind::f16 forms: 24
 *          tensor-core accumulates either way) a tensor-memory accumulator holds before the epilogue
 *          drains it into fp32 registers (default 4); bounds the bias of the tensor core's truncating
 *          accumulate.  1 <= k <= 255.                        */
int gmmnlse_debug_set_tc_chunk(gmmnlse_plan *plan, int k);

/* The nonlinear coupling tensor of Eq. 2 by quadrature, on the GPU:
 *   S_plmn = sum_g F_p F_l F_m F_n dA / sqrt(sum_g F_p^2 dA ... sum_g F_n^2 dA)       [1/m^2]
 * for P real scalar mode fields sampled on G grid points of area dA.  S is the Gram matrix of the P(P+1)/2 pair
 * functions F_p F_l, so the work is one (Q x G)(G x Q) product: it runs on the tcgen05 kind::f16 kernel of a6 with
 * K = G (fp16 hi / lo splits of both operands, two-level accumulation: relative accuracy ~1e-6 of the largest entry);
 * normalisation and expansion to [P]^4 are done in fp64 on the host.
 *   F      HOST [P][G] fp64, any units (the normalisation cancels them);  dA [m^2];
 *   S_out  HOST [P][P][P][P], index ((p*P + l)*P + m)*P + n -- the array gmmnlse_plan_create takes.
 * Runs on the current device and synchronises it.  EINVAL: sizes < 1, NULL pointers, non-finite F, a mode of zero
 * norm; EUNSUPPORTED: G not a multiple of 32.                                                                  */
int gmmnlse_overlap_tensor(int P, long long G, const double *F, double dA, double *S_out);

/* gmmnlse_overlap_tensor for callers that cannot allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same Gram product on the same tcgen05 kernel, but every intermediate lives in
 * ONE static device array of the library (about 4.9 MB, held by every GPU that loads the library until the process
 * exits) instead of per-call cudaMalloc.  The call makes no cudaMalloc / cudaFree / allocating library call, uses no
 * host heap, does not synchronise: all work is enqueued on `stream` (cudaStream_t as void*, NULL = default stream).
 *   F_dev  DEVICE [P][G] fp64 mode fields;  dA [m^2];  S_dev  DEVICE [P][P][P][P] fp64 out (index as S above).
 * Limits: P <= 6, G <= 4096 (e.g. a 64 x 64 grid), G a multiple of 32 -- beyond them EUNSUPPORTED, with the limits
 * spelled out in gmmnlse_last_cuda_error(); gmmnlse_overlap_tensor_noalloc_limits reports them (any pointer may be
 * NULL).  Normalisation happens on the device: F is not checked, a mode of zero norm or a non-finite sample gives
 * non-finite output.  ALL calls on a device share the one array, which keeps the previous call's contents (what must
 * start at zero is cleared by the call): calls that overlap on the GPU -- different streams, or threads -- race;
 * serialise them on one stream.  Runs on the current device; EINVAL: sizes < 1, NULL pointers, dA <= 0.          */
int gmmnlse_overlap_tensor_noalloc(int P, long long G, const double *F_dev, double dA, double *S_dev, void *stream);
int gmmnlse_overlap_tensor_noalloc_limits(int *P_max, long long *G_max, long long *scratch_bytes);

void gmmnlse_plan_destroy(gmmnlse_plan *plan);
const char *gmmnlse_status_string(int status);
const char *gmmnlse_last_cuda_error(void);
int gmmnlse_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GMMNLSE_H_ */
