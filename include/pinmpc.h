/*
 * pinmpc.h — C ABI of libpinmpc.so: batched, construction-free ADMM-MPC solves on one B200 (sm_100a).
 *
 * One handle solves B independent linear time-varying MPC QPs, one per RL environment
 * (eq. (16)-(17), with C = I and X_k = R^nx):
 *
 *     min  sum_{k=0}^{N-1} 1/2 |x_{k+1} - xbar_{k+1}|^2_Q + 1/2 |u_k - ubar_k|^2_R
 *     s.t. x_{k+1} = A_k x_k + B_k u_k + c_k,   x_0 given,   u_k in U_k
 *
 * by a fixed number of scaled-form ADMM iterations in the block order of PAPER.md:L186 eq. (21a)
 * -> (21b) -> (21c): equality-constrained step (exact time-varying LQR, solved with on-chip
 * factors), projection onto U_k, dual update, residuals (the readings of the
 * paper are listed there).  State x = [Theta(3) p(3) omega(3) v(3) g] (nx = 13, BASELINE.json
 * config 0), control u = [f_0..f_{nw-1} | m_0..m_{nw-1} | fh_0..fh_{nf-1}], 3 floats per block.
 *
 * Conventions for every entry point
 *   - plain C types; all array arguments are DEVICE pointers unless the name starts with h_ (host);
 *   - arrays are float32 (contact flags uint8, iteration counts int32), contiguous, env-major,
 *     row-major: [B,N,...] means index ((b*N + k)*... );
 *   - the caller owns all device memory including the workspace; the library owns only the host
 *     context.  Pointers given to pinmpc_set_problem / pinmpc_set_dynamics are BORROWED until the
 *     next set call or pinmpc_destroy;
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  solve/get
 *     enqueue work and return; nothing synchronises the host except pinmpc_create;
 *   - every call returns a pinmpc_status; no exceptions, no abort.  CUDA errors are sticky in the
 *     handle; pinmpc_last_error() describes the last failure;
 *   - a handle is not thread-safe; different handles are independent;
 *   - there is no CPU fallback: a device that is not compute capability 10.x gives
 *     PINMPC_EUNSUPPORTED.
 */
#ifndef PINMPC_H
#define PINMPC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PINMPC_NX 13
#define PINMPC_N_MAX 512
#define PINMPC_SPLIT_N_MAX 1024     /* the stage-local method has no per-horizon on-chip state (N to 400) */

typedef struct pinmpc_ctx *pinmpc_t;

typedef enum {
    PINMPC_OK = 0,
    PINMPC_EINVAL = 1,       /* bad argument (NULL, non-positive size, negative weight ...)         */
    PINMPC_EALLOC = 2,       /* workspace too small or host allocation failed                       */
    PINMPC_ECUDA = 3,        /* a CUDA call or launch failed (sticky)                               */
    PINMPC_ESTATE = 4,       /* call order violated (solve before set_problem, get before solve)    */
    PINMPC_EUNSUPPORTED = 5  /* nx != 13, nu not in {12,18}, N > PINMPC_N_MAX, not an sm_100 device */
} pinmpc_status;

/* Constraint layout: which contacts u holds and the constants of U_k (eq. (7c);
 * BASELINE.json configs 0 and 3).  A foot (6-D wrench contact) in stance is constrained to
 *   |f_x|,|f_y| <= mu f_z,  |m_x| <= mx_coef f_z,  |m_y| <= my_coef f_z,  |m_z| <= mz_coef f_z,
 *   0 <= f_z <= fz_max   — one set, projected jointly; a hand (3-D force contact) in contact to the
 * box |f| <= hand_fmax componentwise; any contact whose flag is 0 to {0}.
 * nu must equal 6*n_wrench + 3*n_force; supported: (2,0) and (2,2). */
typedef struct {
    int n_wrench;
    int n_force;
    float mu, fz_max;
    float mx_coef, my_coef, mz_coef;
    float hand_fmax;
} pinmpc_layout;

/* Solver variants, chosen by measurement.  AUTO picks the structured
 * on-chip solver for problems given by pinmpc_set_problem and the dense one after
 * pinmpc_set_dynamics. */
typedef enum {
    PINMPC_METHOD_AUTO = 0,
    PINMPC_METHOD_DENSE = 1,     /* materialise A_k,B_k,c_k; dense Riccati factors streamed from HBM/L2 */
    PINMPC_METHOD_SRB = 2        /* construction-free structured solver, factors resident on chip       */
} pinmpc_method;

/* Bytes of device workspace pinmpc_create needs for these sizes (0 on invalid arguments). */
size_t pinmpc_workspace_bytes(int nx, int nu, int N, int B, const pinmpc_layout *layout);

/* Same for a specific variant: PINMPC_METHOD_DENSE additionally holds A_k,B_k,c_k and the dense
 * Riccati factors (about 2.7 KB per stage); a workspace of this size enables both variants. */
size_t pinmpc_workspace_bytes_method(int nx, int nu, int N, int B, const pinmpc_layout *layout, pinmpc_method m);

/* Create a handle.  rho > 0 is the ADMM penalty, iters >= 1 the (maximum) iteration count.
 * d_workspace: device memory of at least pinmpc_workspace_bytes(...) bytes, 256-byte aligned,
 * owned by the caller and kept alive until pinmpc_destroy.  Default weights are BASELINE.json's
 * Q = diag(500,500,100,50,50,200,1,1,1,20,20,10,0), R = 1e-5 I and dt = 0.03; change them with
 * pinmpc_set_weights.  Synchronises the device once (to read its properties). */
pinmpc_status pinmpc_create(pinmpc_t *out, int nx, int nu, int N, int B, const pinmpc_layout *layout,
                            float rho, int iters, void *d_workspace, size_t workspace_bytes);

/* Diagonal cost weights (HOST pointers, copied) and the discretisation step of eq. (2)-(4). */
pinmpc_status pinmpc_set_weights(pinmpc_t h, const float *h_Qdiag /*[nx]*/, const float *h_Rdiag /*[nu]*/, float dt);

/* Early exit (north_star (4)).  eps_abs = eps_rel = 0 (default) => exactly `iters` iterations.
 * Otherwise every check_every-th iteration an env stops once
 *   r_prim <= eps_abs + eps_rel max(|u|_inf,|z|_inf)  and  r_dual <= eps_abs + eps_rel rho |y|_inf. */
pinmpc_status pinmpc_set_tolerance(pinmpc_t h, float eps_abs, float eps_rel, int check_every);

/* Warm start of the ADMM iteration (the paper re-solves the MPC at 5-50 Hz inside RL
 * training, so consecutive solves differ by one shifted stage).  d_z0, d_y0: DEVICE arrays
 * [B,N,nu] holding the start values z^0 (constraint copy) and y^0 (scaled dual), e.g. the z, y of the previous
 * solve from pinmpc_get_aux shifted by the caller; borrowed until the next call.  Both NULL (default) = cold
 * start z^0 = y^0 = 0.  The arrays must not alias the library workspace.  One of them NULL: PINMPC_EINVAL. */
pinmpc_status pinmpc_set_warm_start(pinmpc_t h, const float *d_z0, const float *d_y0);

/* Force a solver variant (default PINMPC_METHOD_AUTO). */
pinmpc_status pinmpc_set_method(pinmpc_t h, pinmpc_method m);

/* Tuning knob of the structured solver: envs solved per thread block (1..32; 0 = choose by the
 * occupancy heuristic of DESIGN.md "Kernels"; a value the kernel in use cannot hold falls back to
 * that heuristic).  Results do not depend on it. */
pinmpc_status pinmpc_set_tuning(pinmpc_t h, int envs_per_cta);

/* How the equality step (S3) is parallelised across the horizon (north_star (2); PAPER.md:L206-208 Remark 2,
 * L23): the N stages are cut into `chunks` chunks that are swept concurrently (chunked two-sweep over the
 * time-varying LQR recursion, gains resident in tensor memory).
 *   0 (default) = ceil(N / L) chunks, L = 6 (nu = 12) or 4 (nu = 18), for N >= 16 when the shape fits the chunked
 *                 kernel, else sequential passes (the measured crossover, profiles/r2_sweep_config4.md);
 *   1           = the sequential-pass kernel (two N-step recursions per iteration);
 *   >= 2        = that many chunks; PINMPC_EUNSUPPORTED unless ceil(N / chunks) <= L, chunks <= 128 and
 *                 chunks <= ceil(N / (L - 1)) (room for the chunk operators in the workspace).
 * Results agree to rounding for every setting. */
pinmpc_status pinmpc_set_horizon_chunks(pinmpc_t h, int chunks);

/* Launch shape the last pinmpc_solve of the structured solver used: envs per thread block and horizon
 * chunks (1 = sequential passes).  Either pointer may be NULL.  PINMPC_ESTATE before the first solve. */
pinmpc_status pinmpc_get_launch_shape(pinmpc_t h, int *h_envs_per_cta, int *h_chunks);

/* Per-env problem data, all DEVICE pointers ("{A_k,B_k,e_k} are obtained along the
 * input periodic contact sequence" — here from these raw inputs, on the device, every solve). */
typedef struct {
    const float *x0;           /* [B,nx]      initial state xi_0                                    */
    const float *x_ref;        /* [B,N,nx]    reference xbar_1..xbar_N                              */
    const float *u_ref;        /* [B,N,nu]    reference ubar_0..ubar_{N-1}; NULL => zeros           */
    const uint8_t *contact;    /* [B,N,nc]    1 = contact i active at stage k, nc = n_wrench+n_force */
    const float *foot_r;       /* [B,N,nc,3]  contact position minus CoM, world-aligned axes        */
    const float *yaw;          /* [B,N]       linearisation yaw psi_k                               */
    const float *mass;         /* [B]                                                               */
    const float *inertia;      /* [B,3,3]     body-frame inertia, symmetric positive definite       */
    const float *ext_wrench;   /* [B,N,6]     (F_ext, tau_ext) entering c_k; NULL => c_k = 0        */
} pinmpc_problem;

/* Record the problem (pointers are borrowed, nothing is copied or launched). */
pinmpc_status pinmpc_set_problem(pinmpc_t h, const pinmpc_problem *p);

/* Bypass the dynamics assembly with generic dense LTV matrices (DEVICE pointers, borrowed):
 * A [B,N,nx,nx], Bm [B,N,nx,nu], c [B,N,nx] (NULL => 0).  x0, x_ref, u_ref and contact are still
 * taken from pinmpc_set_problem.  Pass A = NULL to return to on-device assembly.  Solves then use
 * the dense variant. */
pinmpc_status pinmpc_set_dynamics(pinmpc_t h, const float *A, const float *Bm, const float *c);

/* One batched solve: assembly (S1) + factorisation (S2) + iters x (equality step S3, projection
 * S4, dual update S5, residuals / early exit S6), from z = y = 0 or from the values given to pinmpc_set_warm_start.
 * Asynchronous on `stream`. */
pinmpc_status pinmpc_solve(pinmpc_t h, void *stream);

/* Copy results of the last solve into caller DEVICE buffers (any may be NULL), asynchronously on
 * `stream` (use the solve's stream, or order the streams yourself):
 *   x [B,N,nx] = x_1..x_N and u [B,N,nu] = u_0..u_{N-1} of the last equality step (they satisfy
 *   the dynamics exactly), r_prim [B] = max_k |u_k - z_k|_inf, r_dual [B] = rho max_k |z_k -
 *   z_k^prev|_inf, iters_done [B] (int32). */
pinmpc_status pinmpc_get(pinmpc_t h, float *x, float *u, float *r_prim, float *r_dual, int *iters_done, void *stream);

/* The splitting variables after the last solve: z [B,N,nu] (feasible copy), y [B,N,nu] (scaled dual). */
pinmpc_status pinmpc_get_aux(pinmpc_t h, float *z, float *y, void *stream);

/* Receding-horizon shift for the next MPC update (the MPC is re-solved every few control
 * steps): z0[b,k] = z[b,min(k+shift,N-1)] and y0 likewise from the z, y of the last solve (the last stage is
 * repeated), written into caller DEVICE buffers z0, y0 [B,N,nu] that can be handed to pinmpc_set_warm_start.
 * 0 <= shift <= N; asynchronous on `stream` (the solve's stream, or ordered after it).  PINMPC_ESTATE before
 * the first solve and after a pinmpc_set_problem that no solve has followed (shift first, then set the next problem), PINMPC_EINVAL on NULL buffers or a shift out of range. */
pinmpc_status pinmpc_shift_aux(pinmpc_t h, int shift, float *z0, float *y0, void *stream);

/* Materialise the assembled dynamics of the current problem into caller DEVICE buffers
 * A [B,N,nx,nx], Bm [B,N,nx,nu], c [B,N,nx] (any may be NULL); runs the assembly kernel on `stream`. */
pinmpc_status pinmpc_get_dynamics(pinmpc_t h, float *A, float *Bm, float *c, void *stream);

/* Test hook of the product's dynamics assembly (S1, the structured solver never forms A_k, B_k): runs the assembly
 * kernel of the structured solver on the current problem and expands ITS per-stage records (cos/sin of the yaw,
 * I_w, contact offsets, c_k rows, mass) back into dense A [B,N,nx,nx], Bm [B,N,nx,nu] (= E D_k Gh_k, SRB form of
 * PAPER.md:L49-57 eq. (2)-(4)) and c [B,N,nx]; S [B,N,21] is the stored packed upper triangle of
 * S_k = (Bh_k Rt^-1 Bh_k^T)^-1 (Bh_k = rows 6..11 of B_k, Rt = R + rho I) and Tinv [B,N,6] the packed inverse of
 * the Schur complement T_k of the torque block of Gh_k Rt^-1 Gh_k^T.  DEVICE buffers, any may be NULL; asynchronous
 * on `stream`; the workspace's factor arrays are overwritten (call before, not between, solve and get). */
pinmpc_status pinmpc_get_srb_assembly(pinmpc_t h, float *A, float *Bm, float *c, float *S, float *Tinv, void *stream);

/* Number of kernel launches the last pinmpc_solve enqueued (for bench.py's gpu_launches). */
int pinmpc_last_launch_count(pinmpc_t h);

/* Per-kernel timing of the structured solver ("per-phase split (S1, S2, loop)").
 * pinmpc_set_profiling(h, 1) makes every following pinmpc_solve record CUDA events on ITS stream
 * around the three kernels (assembly S1, factorisation S2, iteration S3-S6); 0 turns it off (default).
 * pinmpc_get_kernel_ms synchronises the host on the last recorded event and writes the elapsed
 * milliseconds of the last solve into h_ms[0..2] (HOST array of 3 floats).  PINMPC_ESTATE if
 * profiling is off or no structured solve has been enqueued since it was turned on. */
pinmpc_status pinmpc_set_profiling(pinmpc_t h, int on);
pinmpc_status pinmpc_get_kernel_ms(pinmpc_t h, float *h_ms);

/* ---- Predictive landmarks and the prediction-confidence reward (eq. (10)-(14)) ----
 * Stateless calls on a caller-owned DEVICE ring buffer; all run asynchronously on `stream`.
 *   eq. (10)  n_l = 1 + floor(s_l (N-1))  (float64 product of the float32 s_l), l = 0..n_landmarks-1
 *   eq. (11)  a solve at time t stores (t + n_l, c_hat = x_{n_l}[3:6]) for every landmark
 *   eq. (12)  e_l(t) = c_t - c_hat^{t - n_l}(n_l), omitted when that landmark was never stored
 *   eq. (13)  r_t = exp(-sum_l alpha_l sum_j Qc_j e_{l,j}^2 / sigma_c^2)
 * Time is an integer count of MPC steps per env (int32, restarts with the episode).  The ring holds
 * n_landmarks x (N+1) slots of (c_x, c_y, c_z, target time) per env, addressed by target time modulo N+1;
 * a slot is valid only while its stored target time equals the time asked for. */
#define PINMPC_MAX_LANDMARKS 8
typedef struct {
    int n_landmarks;                      /* N_L in 1..PINMPC_MAX_LANDMARKS                          */
    float s[PINMPC_MAX_LANDMARKS];        /* s_l in [0,1]; the paper sets s_0 = 0, s_{NL-1} = 1        */
    float alpha[PINMPC_MAX_LANDMARKS];    /* prediction-confidence weights, eq. (14)                  */
    float Qc[3];                          /* diagonal of Q_c                                         */
    float sigma_c;                        /* > 0                                                     */
} pinmpc_landmark_cfg;

/* Bytes of the ring buffer for B envs and horizon N (0 on invalid arguments). */
size_t pinmpc_landmark_ring_bytes(int B, int N, const pinmpc_landmark_cfg *cfg);
/* Start of an episode: forget the landmarks of the envs with mask[b] != 0 (DEVICE uint8 [B]; NULL = all). */
pinmpc_status pinmpc_landmark_reset(void *d_ring, int B, int N, const pinmpc_landmark_cfg *cfg, const uint8_t *mask, void *stream);
/* eq. (11): store the landmarks of a solve.  x DEVICE [B,N,13] = x_1..x_N, t DEVICE int32 [B] = solve time. */
pinmpc_status pinmpc_landmark_push(void *d_ring, int B, int N, const pinmpc_landmark_cfg *cfg, const float *x, const int *t, void *stream);
/* The same, reading x straight from the solver's workspace after pinmpc_solve on the same stream (no copy). */
pinmpc_status pinmpc_landmark_push_solver(pinmpc_t h, void *d_ring, const pinmpc_landmark_cfg *cfg, const int *t, void *stream);
/* eq. (12)-(13): c_real DEVICE [B,3] = realised CoM at time t[b]; r DEVICE [B]; n_used DEVICE int32 [B] or NULL
 * = number of landmarks that existed.  Errors: PINMPC_EINVAL on NULL pointers, B,N < 0, n_landmarks out of
 * range or sigma_c <= 0; B = 0 is a no-op. */
pinmpc_status pinmpc_landmark_reward(const void *d_ring, int B, int N, const pinmpc_landmark_cfg *cfg, const float *c_real, const int *t,
                                     float *r, int *n_used, void *stream);

/* ---- The paper's own stage-local ADMM (eq. (18)-(22)): second method -----------------------
 * Velocity form with the lifted state xi_k = [x_k ; u_{k-1}] (n = 13 + nu), copies z_{k+1} = xi_{k+1} and
 * v_k = Bb_k du_k, the dynamics relaxed with a third scaled dual; every update is local to a stage (no recursion
 * over the horizon).  Same QP (16)-(17) as pinmpc_solve, generic dense LTV data.  Per iteration, for every k:
 *   du_k = J_k (v_k - beta_k);  xi_{k+1} = H_k h_k;  gamma_k, gamma~_k;  z_{k+1} = Proj_{R^nx x U_k}((2 gamma~_k +
 *   gamma_k)/3);  v_k = (z_{k+1} + gamma_k)/2;  theta_k, beta_k, lambda_k updates         (eq. (22))
 * with J_k = (Bb_k^T Bb_k)^-1 Bb_k^T and H_k = (Qb + rho I + rho Ab_{k+1}^T Ab_{k+1})^-1 computed once on the
 * device.  All iterates start at 0; `iters` iterations, no acceleration.  Stateless: everything lives in the
 * caller's workspace.  All problem pointers are DEVICE pointers, float32, contiguous. */
typedef struct {
    const float *A;            /* [B,N,13,13]                                                        */
    const float *Bm;           /* [B,N,13,nu]                                                        */
    const float *c;            /* [B,N,13]   offset e_k; NULL => 0                                   */
    const float *x0;           /* [B,13]                                                             */
    const float *u_prev;       /* [B,nu]     u_{-1} of the velocity form; NULL => 0                  */
    const float *x_ref;        /* [B,N,13]   xbar_1..xbar_N                                          */
    const float *u_ref;        /* [B,N,nu]   ubar_0..ubar_{N-1}; NULL => 0                           */
    const uint8_t *contact;    /* [B,N,nc]                                                           */
} pinmpc_split_problem;

/* Bytes of device workspace pinmpc_split_solve needs (0 on unsupported sizes): H_k, G_k and seven lifted vectors
 * per stage, about 4 KB per stage at nu = 12. */
size_t pinmpc_split_workspace_bytes(int nu, int N, int B);

/* Factorise and run `iters` iterations, asynchronously on `stream`.  Outputs (DEVICE, any may be NULL):
 * xi [B,N,13+nu] = xi_1..xi_N = [x_{k+1} ; u_k] of the last (21a) step, z [B,N,13+nu] = the feasible copy,
 * r_prim [B] = max_k |xi_{k+1} - z_{k+1}|_inf of the last iteration.  h_Qdiag [13], h_Rdiag [nu]: HOST.
 * PINMPC_EUNSUPPORTED: nu not in {12,18}, layout not (2,0)/(2,2), N outside 1..PINMPC_SPLIT_N_MAX; PINMPC_EINVAL: NULL
 * required pointer, rho <= 0, iters < 1, negative weight; PINMPC_EALLOC: workspace too small; B = 0: no-op. */
pinmpc_status pinmpc_split_solve(int nu, int N, int B, const pinmpc_layout *layout, const float *h_Qdiag, const float *h_Rdiag,
                                 float rho, int iters, const pinmpc_split_problem *p, void *d_workspace, size_t workspace_bytes,
                                 float *xi, float *z, float *r_prim, void *stream);

/* Options of pinmpc_split_solve_ex.  NULL or all-zero = pinmpc_split_solve.
 *  - Variable scaling x = Sx x~, u = su u~ (PAPER.md:L184 leaves rho and the units open): the iteration (22) runs on
 *    the scaled problem A~ = Sx^-1 A Sx, B~ = su Sx^-1 B, c~ = Sx^-1 c, Q~ = Sx^2 Q, R~ = su^2 R, references and
 *    xi_0 divided by the scales, U~_k = U_k / su (same cone, box bounds divided by su; ONE scalar for all inputs keeps
 *    the projection Euclidean); xi and z are returned in the caller's units, r_prim in the scaled ones.  The limit is
 *    the optimum of the same QP; the iterates differ.
 *  - accel != 0: Nesterov acceleration with restart (PAPER.md:L210 Remark 3; reading: "fast ADMM with restart",
 *    Goldstein et al. 2014) on w = (z, v, theta, beta, lambda): iteration m starts from w^_m and yields w_m;
 *    c_m = rho (|theta_m - theta^_m|^2 + |beta_m - beta^_m|^2 + |lambda_m - lambda^_m|^2 + |dz|^2 + |dv|^2 + |dz - dv|^2)
 *    summed over the env's stages; c_m < eta c_{m-1}: a_{m+1} = (1 + sqrt(1 + 4 a_m^2)) / 2, w^_{m+1} = w_m +
 *    (a_m - 1) / a_{m+1} (w_m - w_{m-1}); else restart: a_{m+1} = 1, w^_{m+1} = w_{m-1}, c_m <- c_{m-1} / eta.
 *    Every env decides for itself.  z is w_M of the last iteration.
 *  - nx, h_x_lo, h_x_hi: the state dimension (all [..,13] shapes of pinmpc_split_problem become [..,nx], xi and z are
 *    [B,N,nx+nu]) and the state box of eq. (17): the projection of (21b) clips the x part of z to it. */
typedef struct {
    const float *h_scale_x;    /* HOST [13] positive, or NULL => 1                                    */
    float scale_u;             /* > 0; 0 => 1                                                         */
    int accel;                 /* 0 plain iteration, 1 accelerated with restart                       */
    float eta;                 /* restart threshold in (0, 1]; 0 => 0.999                             */
    int *d_restarts;           /* DEVICE [B] or NULL: restarts taken per env (accel only)             */
    int nx;                    /* state dimension of A, Bm, c, x0, x_ref: 13 (0 => 13) or 9 (the      */
                               /* centroidal model of eq. (1)-(4)); Qdiag, scale_x, x_lo, x_hi: [nx]  */
    const float *h_x_lo;       /* HOST [nx] or NULL: the state set X_k of eq. (17) as a box on        */
    const float *h_x_hi;       /* xi_{k+1} (caller's units, -INFINITY / INFINITY = free); NULL => R^nx */
} pinmpc_split_options;

/* Workspace of pinmpc_split_solve_ex for these options (scaling adds the scaled problem, about 1.5 KB per stage at
 * nu = 12; acceleration adds two more copies of the five iterate vectors, 1 KB per stage). */
size_t pinmpc_split_workspace_bytes_ex(int nu, int N, int B, const pinmpc_split_options *opts);

/* pinmpc_split_solve with options.  Extra errors: PINMPC_EINVAL for a non-positive or non-finite scale, eta outside
 * (0, 1], x_lo > x_hi; PINMPC_EUNSUPPORTED for nx not in {0, 9, 13}. */
pinmpc_status pinmpc_split_solve_ex(int nu, int N, int B, const pinmpc_layout *layout, const float *h_Qdiag, const float *h_Rdiag,
                                    float rho, int iters, const pinmpc_split_problem *p, const pinmpc_split_options *opts,
                                    void *d_workspace, size_t workspace_bytes, float *xi, float *z, float *r_prim, void *stream);

/* pinmpc_split_solve_ex for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): no workspace argument.  The scratch is a static device array of
 * PINMPC_SPLIT_STATIC_BYTES inside the library: every GPU that loads the library holds it until the process exits.
 * The call allocates nothing (no cudaMalloc / cudaFree / allocating library routine; the array's device address is
 * looked up once per device on the first call there, with the caller's current device).  Same arguments, outputs and
 * errors as pinmpc_split_solve_ex otherwise; PINMPC_EALLOC when pinmpc_split_workspace_bytes_ex(nu, N, B, opts) exceeds
 * PINMPC_SPLIT_STATIC_BYTES (about 3200 stages at nu = 12, 2100 at nu = 18, without options), with the sizes in
 * pinmpc_last_error(NULL).  All calls on a device share the one array: it keeps the last call's contents (everything
 * that must start at zero is cleared on `stream` by the call itself), and two calls that overlap on the GPU (different
 * streams, or different threads) RACE: serialise them. */
#define PINMPC_SPLIT_STATIC_BYTES (16u << 20)
size_t pinmpc_split_static_bytes(void);
pinmpc_status pinmpc_split_solve_static(int nu, int N, int B, const pinmpc_layout *layout, const float *h_Qdiag, const float *h_Rdiag,
                                        float rho, int iters, const pinmpc_split_problem *p, const pinmpc_split_options *opts,
                                        float *xi, float *z, float *r_prim, void *stream);

/* The paper's own 9-state centroidal model (eq. (1)-(4)): xi = [c ; l_G ; k_G] (CoM position, linear
 * and angular centroidal momentum), forward Euler; the lever r_{i,k} = p_{i,k} - c_k of contact i is data.
 * Writes the LTV system of eq. (16), xi_{k+1} = A xi_k + B_k u_k + e:  A [B,N,9,9], Bm [B,N,9,nu], e [B,N,9] with
 * nu = 6 n_wrench + 3 n_force and the input layout above; mass [B], foot_r [B,N,n_wrench+n_force,3]; all DEVICE, float32.
 * Feed them to pinmpc_split_solve_ex with options.nx = 9.  PINMPC_EINVAL: NULL pointer, dt <= 0, no contact; B = 0: no-op. */
pinmpc_status pinmpc_assemble_centroidal(int B, int N, int n_wrench, int n_force, float dt, const float *mass, const float *foot_r,
                                         float *A, float *Bm, float *e, void *stream);

/* Human-readable description of the last error on this handle (owned by the handle; "" if none).
 * With h = NULL: the last pinmpc_create or pinmpc_split_solve_static failure in this thread. */
const char *pinmpc_last_error(pinmpc_t h);

/* Free the host context.  The workspace and all problem buffers stay with the caller. */
void pinmpc_destroy(pinmpc_t h);

#ifdef __cplusplus
}
#endif
#endif /* PINMPC_H */
