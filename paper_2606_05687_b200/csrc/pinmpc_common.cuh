// pinmpc_common.cuh — host context and small device helpers shared by the kernels of libpinmpc.so.
// CUDA path only: nothing here is shared with oracle/ (which is plain C and never includes this).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/pinmpc.h"

#define NX 13
#define NU_MAX 18

// Kernel-side copy of the constraint layout and weights (passed by value as a kernel argument).
struct SolveParams {
    int B, N, nu, nw, nf, iters, check_every;
    float rho, dt, eps_abs, eps_rel;
    float mu, fz_max, cx, cy, cz, hand_fmax;
    float Qd[NX];
    float Rd[NU_MAX];
    // host-computed reciprocals (no divisions in the iteration kernels)
    float tR[NU_MAX];     // 1 / (R_j + rho)
    float rtR[NU_MAX];    // rho / (R_j + rho)
    float iw[5];          // 1 / (mu, mu, cx, cy, cz)
    float phi_inv[3];     // 1 / sum_i tR[f_i axis]  (Lam_FF^-1, the same for every stage)
};

struct ProblemPtrs {
    const float *x0, *x_ref, *u_ref;
    const uint8_t *contact;
    const float *foot_r, *yaw, *mass, *inertia, *ext;
    const float *z0, *y0;      // warm start [B,N,nu] (both NULL: cold start)
};

struct OutPtrs {
    float *x, *u, *z, *y, *r_prim, *r_dual;
    int *iters_done;
};

struct DensePtrs {       // dense variant: materialised dynamics and Riccati factors in HBM
    const float *A, *Bm, *c;          // [B,N,13,13], [B,N,13,nu], [B,N,13] (c may be NULL)
    float *K, *Minv, *s, *kappa;      // [B,N,nu,13], [B,N,nu,nu], [B,N,13], [B,N,nu]
};

// Structured (SRB) variant: per-stage factors kept in the workspace between the assembly,
// factorisation and iteration kernels (st = B*N stages).  "Pass" arrays are env-major and copied
// verbatim into shared memory; "stage" arrays are component-major [comp][st] so that threads
// mapped lane = stage read and write them coalesced.
struct SrbWs {
    float *Kh;     // [st][6][6][2]  gain of the 6-D-input LQR, pairs (Kh[r][j], Kh[r][6+j]), j = 0..5
    float *qv;     // [B][N+1][12]   q_k = Q xbar_k (k = 1..N), q_0 = 0
    float *c6;     // [st][6]        ch = (dt I_w^-1 tau_ext ; dt/m F_ext)   (zeros without ext_wrench)
    float *cs;     // [st][2]        cos, sin of the linearisation yaw
    float *MI;     // [6][st][4]     S_k = D^-1 Lam^-1 D^-1 (packed symmetric, 21 of 24 words): assembly -> factorisation
    // Stage constants streamed by the stage threads of the iteration kernel every iteration: float4
    // component-major, so that thread = stage reads them with coalesced LDG.128 (word w of stage s is
    // at [(w / 4) * st + s] * 4 + w % 4).
    float *RA;     // [7][st][4]     Mh_k^-1 packed symmetric (21) | kg_k = Kh[:,12] x_12 - Mh^-1 hq_k (6) | pad
    float *RB;     // [RBW/4][st][4] T^-1 (6) | I_w (6) | r (3 nc) | Rt^-1 R ubar (nu) | contact bits | pad
};
#define PINMPC_RA_W 28
__host__ __device__ constexpr int pinmpc_rb_width(int nu) { return (12 + 3 * (2 + (nu - 12) / 3) + nu + 1 + 3) & ~3; }
__host__ __device__ inline long pinmpc_rec_index(int w, long st, long s) { return ((long)(w >> 2) * st + s) * 4 + (w & 3); }


struct pinmpc_ctx {
    int nx, nu, N, B;
    pinmpc_layout layout;
    float rho;
    int iters;
    float eps_abs, eps_rel;
    int check_every;
    float Qd[NX], Rd[NU_MAX], dt;
    pinmpc_method method;
    bool have_problem, have_dynamics, solved;
    pinmpc_problem prob;
    const float *userA, *userB, *userC;
    const float *warm_z, *warm_y;
    char *ws;
    size_t ws_bytes;
    // carved from the workspace
    OutPtrs out;
    float *dA, *dB, *dC, *dK, *dMinv, *dS, *dKappa;   // dense-only (NULL when the workspace is the small one)
    SrbWs srb;
    int envs_per_cta;        // tuning knob of the structured solver (0 = auto)
    int chunks;              // horizon chunks of the equality step: 0 = auto, 1 = sequential passes, >= 2 forced
    int psi_cap;             // chunk operators per env the workspace has room for
    float *psi;              // [B][C-2][12][12] chunk operators of the chunked (TMEM) iteration kernel
    int last_G, last_C;      // launch shape of the last structured solve (last_C = 1: sequential passes)
    int sm_count, smem_optin;
    int launch_count;
    int profiling;           // record events around the kernels of the structured solver
    bool prof_valid;
    cudaEvent_t ev[4];
    cudaError_t sticky;
    char err[256];
};

size_t pinmpc_ws_base_bytes(int nu, int N, int B);
size_t pinmpc_ws_dense_bytes(int nu, int N, int B);

// launchers (each returns the number of kernels it enqueued, or -1 with h->err set)
int pinmpc_launch_assemble_dense(pinmpc_ctx *h, float *A, float *Bm, float *c, cudaStream_t st);
int pinmpc_launch_solve_dense(pinmpc_ctx *h, cudaStream_t st);
int pinmpc_launch_solve_srb(pinmpc_ctx *h, cudaStream_t st);
int pinmpc_launch_srb_assembly_debug(pinmpc_ctx *h, float *A, float *Bm, float *c, float *S, float *Tinv, cudaStream_t st);
size_t pinmpc_ws_srb_bytes(int nu, int N, int B);
// chunked, TMEM-resident iteration kernel (pinmpc_tmem.cu)
#define PINMPC_CHUNKED_MIN_N 16     // horizons from which pinmpc_set_horizon_chunks(h, 0) picks the chunked kernel
bool pinmpc_tm_config(const pinmpc_ctx *h, int *G, int *C);
int pinmpc_launch_iterate_tm(pinmpc_ctx *h, int G, int C, cudaStream_t st);
// chunk operators of up to ceil(N / 5) chunks (nu = 12: 5 or 6 stages per chunk), ceil(N / 3) chunks (nu = 18: 3 or 4)
// chunk c of C over N stages (the chunked iteration kernel): the first N % C chunks hold one stage more
__host__ __device__ inline void tm_chunk(int N, int C, int c, int &k0, int &len)
{
    const int base = N / C, rem = N - base * C;
    k0 = c * base + (c < rem ? c : rem);
    len = base + (c < rem ? 1 : 0);
}

void pinmpc_note_error(const char *msg);   // pinmpc_api.cu: sets what pinmpc_last_error(NULL) returns in this thread
inline int pinmpc_psi_cap(int N, int nu) { int c = (nu == 12 ? (N + 4) / 5 : (N + 2) / 3) - 2; return c > 0 ? c : 0; }

static inline SolveParams make_params(const pinmpc_ctx *h)
{
    SolveParams p;
    memset(&p, 0, sizeof p);
    p.B = h->B; p.N = h->N; p.nu = h->nu; p.nw = h->layout.n_wrench; p.nf = h->layout.n_force;
    p.iters = h->iters; p.check_every = h->check_every;
    p.rho = h->rho; p.dt = h->dt; p.eps_abs = h->eps_abs; p.eps_rel = h->eps_rel;
    p.mu = h->layout.mu; p.fz_max = h->layout.fz_max; p.cx = h->layout.mx_coef; p.cy = h->layout.my_coef;
    p.cz = h->layout.mz_coef; p.hand_fmax = h->layout.hand_fmax;
    for (int i = 0; i < NX; i++) p.Qd[i] = h->Qd[i];
    for (int i = 0; i < NU_MAX; i++) {
        p.Rd[i] = h->Rd[i];
        p.tR[i] = 1.0f / (h->Rd[i] + h->rho);
        p.rtR[i] = h->rho / (h->Rd[i] + h->rho);
    }
    p.iw[0] = p.iw[1] = 1.0f / p.mu; p.iw[2] = 1.0f / p.cx; p.iw[3] = 1.0f / p.cy; p.iw[4] = 1.0f / p.cz;
    for (int a = 0; a < 3; a++) {
        float sum = 0.0f;
        for (int i = 0; i < p.nw + p.nf; i++) sum += p.tR[(i < p.nw ? 3 * i : 6 * p.nw + 3 * (i - p.nw)) + a];
        p.phi_inv[a] = 1.0f / sum;
    }
    return p;
}

static inline ProblemPtrs make_problem_ptrs(const pinmpc_ctx *h)
{
    ProblemPtrs q;
    q.x0 = h->prob.x0; q.x_ref = h->prob.x_ref; q.u_ref = h->prob.u_ref; q.contact = h->prob.contact;
    q.foot_r = h->prob.foot_r; q.yaw = h->prob.yaw; q.mass = h->prob.mass; q.inertia = h->prob.inertia;
    q.ext = h->prob.ext_wrench;
    q.z0 = h->warm_z; q.y0 = h->warm_y;
    return q;
}

#ifdef __CUDACC__
// ---------------------------------------------------------------------------------------------
// device helpers
// ---------------------------------------------------------------------------------------------
// Inverse of a 3x3 matrix (adjugate / determinant), row-major.
__device__ __forceinline__ void inv3f(const float *M, float *Mi)
{
    float c00 = M[4] * M[8] - M[5] * M[7], c01 = M[5] * M[6] - M[3] * M[8], c02 = M[3] * M[7] - M[4] * M[6];
    float id = 1.0f / (M[0] * c00 + M[1] * c01 + M[2] * c02);
    Mi[0] = c00 * id; Mi[1] = (M[2] * M[7] - M[1] * M[8]) * id; Mi[2] = (M[1] * M[5] - M[2] * M[4]) * id;
    Mi[3] = c01 * id; Mi[4] = (M[0] * M[8] - M[2] * M[6]) * id; Mi[5] = (M[2] * M[3] - M[0] * M[5]) * id;
    Mi[6] = c02 * id; Mi[7] = (M[1] * M[6] - M[0] * M[7]) * id; Mi[8] = (M[0] * M[4] - M[1] * M[3]) * id;
}

// I_w^{-1} = R_z(yaw) I_b^{-1} R_z(yaw)^T  (BASELINE.json config 0), row-major 3x3.
__device__ __forceinline__ void world_inertia_inv(const float *Ibinv, float cs, float sn, float *W)
{
    // T = R_z Ibinv
    float T[9];
#pragma unroll
    for (int j = 0; j < 3; j++) {
        T[0 * 3 + j] = cs * Ibinv[0 * 3 + j] - sn * Ibinv[1 * 3 + j];
        T[1 * 3 + j] = sn * Ibinv[0 * 3 + j] + cs * Ibinv[1 * 3 + j];
        T[2 * 3 + j] = Ibinv[2 * 3 + j];
    }
    // W = T R_z^T : W[i][0] = T[i][0] c - T[i][1] s ; W[i][1] = T[i][0] s + T[i][1] c ; W[i][2] = T[i][2]
#pragma unroll
    for (int i = 0; i < 3; i++) {
        W[i * 3 + 0] = T[i * 3 + 0] * cs - T[i * 3 + 1] * sn;
        W[i * 3 + 1] = T[i * 3 + 0] * sn + T[i * 3 + 1] * cs;
        W[i * 3 + 2] = T[i * 3 + 2];
    }
}

// Free minimiser t* of  1/2 (t-t0)^2 + 1/2 sum_i (a_i - w_i t)_+^2  (a_i = |y_i| >= 0): the height
// of the exact Euclidean projection onto the foot wrench set before clamping to [0, f_max]
// (z-update).  The derivative g(t) is increasing, concave and
// piecewise linear with kinks b_i = a_i / w_i, so coordinate i is clipped at the optimum
// (a_i > w_i t*) exactly when g(b_i) > 0.  Five kink evaluations decide the clipped set, one
// division gives t*.  Branch-free; w_i > 0 required (iw_i = 1 / w_i).
__device__ __forceinline__ float wrench_height(float t0, const float a[5], const float w[5], const float iw[5])
{
    float num = t0, den = 1.0f;
#pragma unroll
    for (int i = 0; i < 5; i++) {
        float bi = a[i] * iw[i];
        float g = bi - t0;
#pragma unroll
        for (int j = 0; j < 5; j++)
            if (j != i) g -= w[j] * fmaxf(a[j] - w[j] * bi, 0.0f);
        if (g > 0.0f) { num = fmaf(w[i], a[i], num); den = fmaf(w[i], w[i], den); }
    }
    return __fdividef(num, den);                     // den in [1, 1 + sum w_i^2]: the 2-ulp approximate division is safe
}

// Exact projection of one foot wrench (f, m) onto W; writes the projected 6 values.
__device__ __forceinline__ void project_wrench(const SolveParams &P, float fx, float fy, float fz, float mx, float my,
                                               float mz, float &ofx, float &ofy, float &ofz, float &omx, float &omy,
                                               float &omz)
{
    const float w[5] = { P.mu, P.mu, P.cx, P.cy, P.cz };
    const float iw[5] = { P.iw[0], P.iw[1], P.iw[2], P.iw[3], P.iw[4] };
    const float a[5] = { fabsf(fx), fabsf(fy), fabsf(mx), fabsf(my), fabsf(mz) };
    float t = wrench_height(fz, a, w, iw);
    t = fminf(fmaxf(t, 0.0f), P.fz_max);
    ofx = copysignf(fminf(a[0], w[0] * t), fx);
    ofy = copysignf(fminf(a[1], w[1] * t), fy);
    ofz = t;
    omx = copysignf(fminf(a[2], w[2] * t), mx);
    omy = copysignf(fminf(a[3], w[3] * t), my);
    omz = copysignf(fminf(a[4], w[4] * t), mz);
}

__device__ __forceinline__ float warp_max(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
#endif  // __CUDACC__
