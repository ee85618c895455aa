// The paper's own stage-local ADMM (pi^n MPC proper), eq. (18)-(22); SURVEY 8(f) rank 1.
// Second method next to the exact-dynamics solver: no recursion over the horizon, every update is local to a
// stage and reads at most the neighbouring stage.  Generic dense LTV data (A_k, B_k, c_k), nx = 13 (the SRB model)
// or nx = 9 (the paper's centroidal model, eq. (1)-(4)); a box X_k on the states (eq. (17)) is part of the projection.
//
// Lifted state xi_k = [x_k ; u_{k-1}] (n = 13 + nu <= 31), Ab = [[A, B],[0, I]], Bb = [B ; I], eb = [c ; 0].
// One warp per stage, lane i = component i of the lifted vectors; matrices are read so that consecutive lanes
// touch consecutive words (H and G are symmetric, so "column i" is read as row-major [j][i]).
//   k_split_factor  G_k = (B_k^T B_k + I)^-1 (J_k = G_k Bb_k^T), H_k = (Qb + rho I + rho Ab_{k+1}^T Ab_{k+1})^-1 (both SPD:
//                   Gauss-Jordan without pivoting, rows in registers, pivot row broadcast by shuffles) and
//                   [A_k B_k]^T for the coalesced row reads of (21b)
//   k_split_a       (21a): du_k = J_k (v_k - beta_k), xi_{k+1} = H_k h_k from the previous z, v, theta, beta, lambda
//   k_split_b       (21b), (21c): gamma, gamma~, z = Proj((2 gamma~ + gamma)/3), v = (z + gamma)/2, dual updates
// The factors stream from HBM every iteration (about 8.1 KB per stage-iteration at nu = 12): the method is
// reported against the HBM roofline.
//
// pinmpc_split_solve_ex adds (oracle/split.py header):
//   variable scaling   x = Sx x~, u = su u~: k_split_scale writes the scaled problem (A~ = Sx^-1 A Sx, B~ = su Sx^-1 B,
//                      c~, references, xi_0) into the workspace once, Q~ = Sx^2 Q, R~ = su^2 R and the box bounds of
//                      the wrench set / su go into the parameters, k_split_unscale scales xi and z back
//   fast ADMM with restart on w = (z, v, theta, beta, lambda): (21a)/(21b) read the extrapolated point w^, (21b)
//                      writes w_m into a ring of two buffers and the stage's share of the combined residual c_m;
//                      k_split_decide (one thread per env, stages summed in order in double: deterministic) takes
//                      the accept / restart decision, k_split_extrapolate forms w^_{m+1}
#include "pinmpc_common.cuh"
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <mutex>

namespace {

constexpr unsigned FULL = 0xffffffffu;
constexpr int SPLIT_WARPS = 8;
constexpr int NW_FEET = 2;              // 6-D wrench contacts (supported layouts: (2,0) and (2,2))

struct SplitPtrs {
    const float *A, *Bm, *c, *x0, *u_prev, *x_ref, *u_ref;
    const uint8_t *contact;
    float *H, *G;                          // [st][n][n], [st][nu][nu]
    float *Tt;                             // [st][n][13]  [A_k B_k] transposed: column-major rows for coalesced reads in (21b)
    float *xi, *du;                        // [st][n], [st][nu]
    const float *z, *v, *th, *be, *la;     // [st][n] the point the iteration starts from (w^ with acceleration)
    float *nz, *nv, *nth, *nbe, *nla;      // [st][n] the point it produces (the same buffers without acceleration)
    float *rs;                             // [st] per-stage primal residual of the last iteration
    float *cpart;                          // [st] per-stage share of the combined residual c_m (acceleration) or NULL
    float x_lo[NX], x_hi[NX];              // the state box X_k in scaled units (+-inf = free)
};

struct SplitScale { float sx[NX], isx[NX], su, isu; };

// In-place Gauss-Jordan inverse of an SPD m x m matrix without pivoting: lane i holds row i in registers
// (lanes >= m hold zero rows), the pivot row is broadcast with shuffles; everything is unrolled, so the rows
// never leave the register file.
template <int m> __device__ __forceinline__ void spd_inverse_regs(float (&row)[m], int lane)
{
#pragma unroll
    for (int p = 0; p < m; p++) {
        const float d = 1.0f / __shfl_sync(FULL, row[p], p);
        const float f = row[p];                                  // M[lane][p] before this pivot
#pragma unroll
        for (int j = 0; j < m; j++) {
            const float pj = __shfl_sync(FULL, row[j], p);
            const float rpj = (j == p) ? d : pj * d;             // the scaled pivot row
            row[j] = (lane == p) ? rpj : ((j == p) ? -f * d : fmaf(-f, rpj, row[j]));
        }
    }
}

template <int NXT, int NU>
__global__ void __launch_bounds__(SPLIT_WARPS * 32) k_split_factor(SolveParams P, SplitPtrs q)
{
    constexpr int n = NXT + NU;
    __shared__ float sT[SPLIT_WARPS][NXT * n];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const long s = (long)blockIdx.x * SPLIT_WARPS + wib, st = (long)P.B * P.N;
    if (s >= st) return;
    const int k = (int)(s % P.N);
    float *T = sT[wib];
    // ---- G = (B^T B + I)^-1 : B_k staged in shared memory, lane i keeps column i
    {
        const float *Bk = q.Bm + s * NXT * NU;
        for (int i = lane; i < NXT * NU; i += 32) T[i] = Bk[i];
        __syncwarp();
        const int lu = lane < NU ? lane : 0;
        float col[NXT], g[NU];
#pragma unroll
        for (int a = 0; a < NXT; a++) col[a] = lane < NU ? T[a * NU + lu] : 0.0f;
#pragma unroll
        for (int j = 0; j < NU; j++) {
            float acc = lane == j ? 1.0f : 0.0f;
#pragma unroll
            for (int a = 0; a < NXT; a++) acc = fmaf(col[a], T[a * NU + j], acc);
            g[j] = acc;
        }
        spd_inverse_regs<NU>(g, lane);
        if (lane < NU) {
#pragma unroll
            for (int j = 0; j < NU; j++) q.G[s * NU * NU + j * NU + lane] = g[j];
        }
        __syncwarp();
    }
    // ---- Tt_k = [A_k B_k]^T for (21b)
    {
        const float *Ak = q.A + s * NXT * NXT, *Bk = q.Bm + s * NXT * NU;
        for (int i = lane; i < NXT * n; i += 32) {
            const int a = i / n, j = i - a * n;
            T[i] = j < NXT ? Ak[a * NXT + j] : Bk[a * NU + j - NXT];
        }
        __syncwarp();
        for (int i = lane; i < NXT * n; i += 32) {
            const int c = i / NXT, r = i - c * NXT;
            q.Tt[s * NXT * n + i] = T[r * n + c];
        }
        __syncwarp();
    }
    // ---- H = (Qb + rho I [+ rho Ab_{k+1}^T Ab_{k+1}])^-1 ;  Ab^T Ab = T^T T + [[0, 0],[0, I]],  T = [A_{k+1} B_{k+1}] (13 x n)
    const bool nxt = k < P.N - 1;
    if (nxt) {
        const float *A1 = q.A + (s + 1) * NXT * NXT, *B1 = q.Bm + (s + 1) * NXT * NU;
        for (int i = lane; i < NXT * n; i += 32) {
            const int a = i / n, j = i - a * n;
            T[i] = j < NXT ? A1[a * NXT + j] : B1[a * NU + j - NXT];
        }
    }
    __syncwarp();
    const int ln = lane < n ? lane : 0;
    const float qd = lane < NXT ? P.Qd[lane] : (lane < n ? P.Rd[lane - NXT] : 0.0f);
    float h[n], col[NXT];
#pragma unroll
    for (int a = 0; a < NXT; a++) col[a] = (nxt && lane < n) ? T[a * n + ln] : 0.0f;
#pragma unroll
    for (int j = 0; j < n; j++) {
        float acc = (lane == j && lane >= NXT && nxt) ? 1.0f : 0.0f;
        if (nxt) {
#pragma unroll
            for (int a = 0; a < NXT; a++) acc = fmaf(col[a], T[a * n + j], acc);
        }
        h[j] = fmaf(P.rho, acc, lane == j ? qd + P.rho : 0.0f);
    }
    spd_inverse_regs<n>(h, lane);
    if (lane < n) {
#pragma unroll
        for (int j = 0; j < n; j++) q.H[s * n * n + j * n + lane] = h[j];
    }
}

// (21a)
template <int NXT, int NU>
__global__ void __launch_bounds__(SPLIT_WARPS * 32, 5) k_split_a(SolveParams P, SplitPtrs q)
{
    constexpr int n = NXT + NU;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const long s = (long)blockIdx.x * SPLIT_WARPS + wib, st = (long)P.B * P.N;
    if (s >= st) return;
    const int k = (int)(s % P.N);
    const bool on = lane < n, isx = lane < NXT;
    const int ju = isx ? 0 : (on ? lane - NXT : 0);
    // The kernel is bound by memory latency, so the matrix elements a lane needs (column `lane` of B_k, G_k,
    // Ab_{k+1}, H_k) are requested in batches of independent loads before they are used.
    const bool nxt = k < P.N - 1;
    const long s1 = nxt ? s + 1 : s;
    const float *Bk = q.Bm + s * NXT * NU, *Gk = q.G + s * NU * NU, *Hk = q.H + s * n * n;
    const float *A1 = q.A + s1 * NXT * NXT, *B1 = q.Bm + s1 * NXT * NU;
    const int lu = lane < NU ? lane : 0, ln = on ? lane : 0;
    float bb[NXT], gb[NU];
#pragma unroll
    for (int a = 0; a < NXT; a++) bb[a] = Bk[a * NU + lu];
#pragma unroll
    for (int l = 0; l < NU; l++) gb[l] = Gk[l * NU + lu];
    const float vv = on ? q.v[s * n + lane] : 0.0f, bv = on ? q.be[s * n + lane] : 0.0f;
    const float zv = on ? q.z[s * n + lane] : 0.0f, tv = on ? q.th[s * n + lane] : 0.0f;
    float w = 0.0f;
    if (on && nxt) {
        w = q.z[s1 * n + lane] - q.v[s1 * n + lane] + q.la[s1 * n + lane];
        if (isx && q.c) w -= q.c[s1 * NXT + lane];
    }
    const float ref = on ? (isx ? q.x_ref[s * NXT + lane] : (q.u_ref ? q.u_ref[s * NU + ju] : 0.0f)) : 0.0f;
    // du = G (B^T r_x + r_u),  r = v - beta
    const float r = vv - bv;
    float t = __shfl_sync(FULL, r, NXT + lu);                               // r_u[lane] on lanes < NU
#pragma unroll
    for (int a = 0; a < NXT; a++) t = fmaf(bb[a], __shfl_sync(FULL, r, a), t);
    float ab[NXT];
#pragma unroll
    for (int a = 0; a < NXT; a++) ab[a] = isx ? A1[a * NXT + lane] : B1[a * NU + ju];
    float du = 0.0f;
#pragma unroll
    for (int l = 0; l < NU; l++) du = fmaf(gb[l], __shfl_sync(FULL, t, l), du);
    if (lane < NU) q.du[s * NU + lane] = du;
    constexpr int H1 = (n + 1) / 2;
    float ha[H1];
#pragma unroll
    for (int j = 0; j < H1; j++) ha[j] = Hk[j * n + ln];
    // h = qb + rho (z - theta) + rho Ab_{k+1}^T (z_{k+1} - v_{k+1} - eb_{k+1} + lam_{k+1})
    float h = 0.0f;
    if (on) h = fmaf(P.rho, zv - tv, (isx ? P.Qd[lane] : P.Rd[ju]) * ref);
    if (nxt) {
        float acc = isx ? 0.0f : w;
#pragma unroll
        for (int a = 0; a < NXT; a++) acc = fmaf(ab[a], __shfl_sync(FULL, w, a), acc);
        if (on) h = fmaf(P.rho, acc, h);
    }
    float hb[n - H1];
#pragma unroll
    for (int j = H1; j < n; j++) hb[j - H1] = Hk[j * n + ln];
    // xi = H h
    float xi = 0.0f;
#pragma unroll
    for (int j = 0; j < H1; j++) xi = fmaf(ha[j], __shfl_sync(FULL, h, j), xi);
#pragma unroll
    for (int j = H1; j < n; j++) xi = fmaf(hb[j - H1], __shfl_sync(FULL, h, j), xi);
    if (on) q.xi[s * n + lane] = xi;
}

// (21b), (21c)
template <int NXT, int NU>
__global__ void __launch_bounds__(SPLIT_WARPS * 32) k_split_b(SolveParams P, SplitPtrs q, int last)
{
    constexpr int n = NXT + NU, NC = 2 + (NU - 12) / 3;
    __shared__ float su[SPLIT_WARPS][NU_MAX + 2];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const long s = (long)blockIdx.x * SPLIT_WARPS + wib, st = (long)P.B * P.N;
    if (s >= st) return;
    const long b = s / P.N;
    const int k = (int)(s - b * P.N);
    const bool on = lane < n, isx = lane < NXT;
    const int ju = isx ? 0 : (on ? lane - NXT : 0);
    const float *Tt = q.Tt + s * NXT * n + (isx ? lane : 0);      // column-major [A_k B_k]: Tt[a * 13 + row]
    // xi_k (the lifted state entering stage k): data for k = 0
    float xp = 0.0f;
    if (on) {
        if (k == 0) xp = isx ? q.x0[b * NXT + lane] : (q.u_prev ? q.u_prev[b * NU + ju] : 0.0f);
        else xp = q.xi[(s - 1) * n + lane];
    }
    const float du = (on && !isx) ? q.du[s * NU + ju] : 0.0f;
    // Ab xi_k and Bb du
    float Axi = isx ? 0.0f : xp, Bdu = isx ? 0.0f : du;
#pragma unroll
    for (int a = 0; a < n; a++) {
        const float xa = __shfl_sync(FULL, xp, a);
        if (isx) Axi = fmaf(Tt[a * NXT], xa, Axi);
    }
#pragma unroll
    for (int j = 0; j < NU; j++) {
        const float dj = __shfl_sync(FULL, du, NXT + j);
        if (isx) Bdu = fmaf(Tt[(NXT + j) * NXT], dj, Bdu);
    }
    float xi = 0.0f, th = 0.0f, be = 0.0f, la = 0.0f, e = 0.0f;
    if (on) {
        xi = q.xi[s * n + lane]; th = q.th[s * n + lane]; be = q.be[s * n + lane]; la = q.la[s * n + lane];
        if (isx && q.c) e = q.c[s * NXT + lane];
    }
    const float gamma = Bdu + be - Axi - e + la;
    const float gammat = xi + th + Axi + e - la;
    const float w = (2.0f * gammat + gamma) * (1.0f / 3.0f);
    // projection of the u part onto U_k (the x part is free): through shared memory, one lane per contact
    float *uw = su[wib];
    if (on && !isx) uw[ju] = w;
    __syncwarp();
    if (lane < NC) {
        const bool in_contact = q.contact[s * NC + lane] != 0;
        if (lane < NW_FEET) {
            const int f0 = 3 * lane, m0 = 3 * NW_FEET + 3 * lane;
            float o[6] = { 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f };
            if (in_contact) project_wrench(P, uw[f0], uw[f0 + 1], uw[f0 + 2], uw[m0], uw[m0 + 1], uw[m0 + 2], o[0], o[1], o[2], o[3], o[4], o[5]);
            uw[f0] = o[0]; uw[f0 + 1] = o[1]; uw[f0 + 2] = o[2]; uw[m0] = o[3]; uw[m0 + 1] = o[4]; uw[m0 + 2] = o[5];
        } else {
            const int f0 = 6 * NW_FEET + 3 * (lane - NW_FEET);
#pragma unroll
            for (int a = 0; a < 3; a++) uw[f0 + a] = in_contact ? fminf(fmaxf(uw[f0 + a], -P.hand_fmax), P.hand_fmax) : 0.0f;
        }
    }
    __syncwarp();
    const float z = isx ? fminf(fmaxf(w, q.x_lo[isx ? lane : 0]), q.x_hi[isx ? lane : 0]) : (on ? uw[ju] : 0.0f);      // X_k: a box (+-inf = free)
    const float v = 0.5f * (z + gamma);
    if (q.cpart) {
        // c_m share of this stage: rho (|d theta|^2 + |d beta|^2 + |d lambda|^2 + |dz|^2 + |dv|^2 + |dz - dv|^2) against w^
        float cs = 0.0f;
        if (on) {
            const float dth = xi - z, dbe = Bdu - v, dla = z - Axi - v - e;
            const float dz = z - q.z[s * n + lane], dv = v - q.v[s * n + lane];
            cs = dth * dth + dbe * dbe + dla * dla + dz * dz + dv * dv + (dz - dv) * (dz - dv);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) cs += __shfl_xor_sync(FULL, cs, o);
        if (lane == 0) q.cpart[s] = P.rho * cs;
    }
    if (on) {
        q.nz[s * n + lane] = z;
        q.nv[s * n + lane] = v;
        q.nth[s * n + lane] = th + xi - z;
        q.nbe[s * n + lane] = be + Bdu - v;
        q.nla[s * n + lane] = la + z - Axi - v - e;
    }
    if (last) {
        const float rmax = warp_max(on ? fabsf(xi - z) : 0.0f);
        if (lane == 0) q.rs[s] = rmax;
    }
}

// x = Sx x~, u = su u~: the scaled problem, written once.  One thread per element of the largest array (A or B).
__global__ void k_split_scale(int B, int N, int nx, int nu, SplitScale S, const float *A, const float *Bm, const float *c, const float *x0,
                              const float *u_prev, const float *x_ref, const float *u_ref, float *sA, float *sB, float *sc, float *sx0,
                              float *sup, float *sxr, float *sur)
{
    const long st = (long)B * N, i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < st * nx * nx) { const int r = (int)((i / nx) % nx), col = (int)(i % nx); sA[i] = A[i] * S.isx[r] * S.sx[col]; }
    if (i < st * nx * nu) { const int r = (int)((i / nu) % nx); sB[i] = Bm[i] * S.isx[r] * S.su; }
    if (i < st * nx) { const int r = (int)(i % nx); if (c) sc[i] = c[i] * S.isx[r]; sxr[i] = x_ref[i] * S.isx[r]; }
    if (i < st * nu && u_ref) sur[i] = u_ref[i] * S.isu;
    if (i < (long)B * nx) sx0[i] = x0[i] * S.isx[(int)(i % nx)];
    if (i < (long)B * nu && u_prev) sup[i] = u_prev[i] * S.isu;
}

__global__ void k_split_unscale(long st, int nx, int n, SplitScale S, const float *in, float *out)
{
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= st * n) return;
    const int j = (int)(i % n);
    out[i] = in[i] * (j < nx ? S.sx[j] : S.su);
}

// Accept / restart decision of iteration m for every env (oracle/split.py header).  acc[b] = (alpha, c_prev, mom, restart).
__global__ void k_split_decide(int B, int N, float eta, const float *cpart, float4 *acc, int *restarts)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    double c = 0.0;
    for (int k = 0; k < N; k++) c += (double)cpart[(long)b * N + k];
    float4 a = acc[b];
    const float cm = (float)c;
    if (cm < eta * a.y) {
        const float an = 0.5f * (1.0f + sqrtf(1.0f + 4.0f * a.x * a.x));
        a.z = (a.x - 1.0f) / an; a.x = an; a.y = cm; a.w = 0.0f;
    } else {
        a.z = 0.0f; a.x = 1.0f; a.y = a.y / eta; a.w = 1.0f;
        if (restarts) restarts[b] += 1;
    }
    acc[b] = a;
}

// w^_{m+1} = w_m + mom (w_m - w_{m-1}), or w_{m-1} after a restart; the five vectors z, v, theta, beta, lambda are
// contiguous [5][st][n] in each buffer.
__global__ void k_split_extrapolate(long st, int N, int n, const float4 *acc, const float *wm, const float *wp, float *hat)
{
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 5 * st * n) return;
    const long s = (i % (st * n)) / n;
    const float4 a = acc[s / N];
    const float m = wm[i], p = wp[i];
    hat[i] = a.w != 0.0f ? p : fmaf(a.z, m - p, m);
}

__global__ void k_split_accel_init(int B, float4 *acc, int *restarts)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    acc[b] = make_float4(1.0f, __int_as_float(0x7f800000), 0.0f, 0.0f);
    if (restarts) restarts[b] = 0;
}

__global__ void k_split_residual(const float *rs, float *r_prim, int B, int N)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    float m = 0.0f;
    for (int k = 0; k < N; k++) m = fmaxf(m, rs[(long)b * N + k]);
    r_prim[b] = m;
}

size_t split_floats(int nx, int nu, long st)
{
    const long n = nx + nu;
    return (size_t)st * (n * n + nu * nu + nx * n + 7 * n + nu + 1);
}

bool opt_scaled(const pinmpc_split_options *o) { return o && (o->h_scale_x != nullptr || (o->scale_u != 0.0f && o->scale_u != 1.0f)); }
bool opt_accel(const pinmpc_split_options *o) { return o && o->accel != 0; }

int opt_nx(const pinmpc_split_options *o) { return (o && o->nx != 0) ? o->nx : NX; }

size_t split_floats_ex(int nu, long st, long B, const pinmpc_split_options *o)
{
    const long nx = opt_nx(o), n = nx + nu;
    size_t f = split_floats((int)nx, nu, st);
    if (opt_scaled(o)) f += (size_t)st * (nx * nx + nx * nu + 2 * nx + nu) + (size_t)B * n;
    if (opt_accel(o)) f += (size_t)st * (10 * n + 1) + (size_t)B * 4 + 4;
    return f;
}

template <int NXT, int NU>
pinmpc_status run(const SolveParams &P, SplitPtrs q, int iters, float *r_prim, bool accel, float eta, float *w1, float *hat, float4 *acc,
                  int *restarts, cudaStream_t stream)
{
    constexpr int n = NXT + NU;
    const long st = (long)P.B * P.N;
    const unsigned blocks = (unsigned)((st + SPLIT_WARPS - 1) / SPLIT_WARPS);
    k_split_factor<NXT, NU><<<blocks, SPLIT_WARPS * 32, 0, stream>>>(P, q);
    float *w0 = q.nz;                                        // ring buffer 0 = the plain iteration's z, v, theta, beta, lambda
    if (accel) {
        k_split_accel_init<<<(P.B + 127) / 128, 128, 0, stream>>>(P.B, acc, restarts);
        q.z = hat; q.v = hat + st * n; q.th = hat + 2 * st * n; q.be = hat + 3 * st * n; q.la = hat + 4 * st * n;
    }
    for (int it = 0; it < iters; it++) {
        if (accel) {
            float *wm = (it & 1) ? w1 : w0;
            q.nz = wm; q.nv = wm + st * n; q.nth = wm + 2 * st * n; q.nbe = wm + 3 * st * n; q.nla = wm + 4 * st * n;
        }
        k_split_a<NXT, NU><<<blocks, SPLIT_WARPS * 32, 0, stream>>>(P, q);
        k_split_b<NXT, NU><<<blocks, SPLIT_WARPS * 32, 0, stream>>>(P, q, it == iters - 1 && r_prim != nullptr);
        if (accel && it < iters - 1) {
            k_split_decide<<<(P.B + 127) / 128, 128, 0, stream>>>(P.B, P.N, eta, q.cpart, acc, restarts);
            const long tot = 5 * st * n;
            k_split_extrapolate<<<(unsigned)((tot + 255) / 256), 256, 0, stream>>>(st, P.N, n, acc, (it & 1) ? w1 : w0, (it & 1) ? w0 : w1, hat);
        }
    }
    if (r_prim) k_split_residual<<<(P.B + 127) / 128, 128, 0, stream>>>(q.rs, r_prim, P.B, P.N);
    return cudaGetLastError() == cudaSuccess ? PINMPC_OK : PINMPC_ECUDA;
}

}   // namespace

extern "C" size_t pinmpc_split_workspace_bytes_ex(int nu, int N, int B, const pinmpc_split_options *opts)
{
    if ((nu != 12 && nu != 18) || N < 1 || N > PINMPC_SPLIT_N_MAX || B < 0) return 0;
    if (opt_nx(opts) != NX && opt_nx(opts) != 9) return 0;
    return split_floats_ex(nu, (long)B * N, B, opts) * sizeof(float) + 256;
}

extern "C" size_t pinmpc_split_workspace_bytes(int nu, int N, int B) { return pinmpc_split_workspace_bytes_ex(nu, N, B, nullptr); }

extern "C" pinmpc_status pinmpc_split_solve_ex(int nu, int N, int B, const pinmpc_layout *layout, const float *h_Qdiag, const float *h_Rdiag,
                                               float rho, int iters, const pinmpc_split_problem *p, const pinmpc_split_options *opts,
                                               void *d_ws, size_t ws_bytes, float *xi, float *z, float *r_prim, void *stream)
{
    if ((nu != 12 && nu != 18) || N < 1 || N > PINMPC_SPLIT_N_MAX) return PINMPC_EUNSUPPORTED;
    if (!layout || layout->n_wrench != 2 || 6 * layout->n_wrench + 3 * layout->n_force != nu) return PINMPC_EUNSUPPORTED;
    if (B < 0 || !(rho > 0.0f) || iters < 1 || !h_Qdiag || !h_Rdiag || !p) return PINMPC_EINVAL;
    const int nx = opt_nx(opts);
    if (nx != NX && nx != 9) return PINMPC_EUNSUPPORTED;
    const bool scaled = opt_scaled(opts), accel = opt_accel(opts);
    SplitScale S;
    for (int i = 0; i < NX; i++) {
        const float v = (opts && opts->h_scale_x && i < nx) ? opts->h_scale_x[i] : 1.0f;
        if (!(v > 0.0f) || !std::isfinite(v)) return PINMPC_EINVAL;
        S.sx[i] = v; S.isx[i] = 1.0f / v;
    }
    S.su = (opts && opts->scale_u != 0.0f) ? opts->scale_u : 1.0f;
    if (!(S.su > 0.0f) || !std::isfinite(S.su)) return PINMPC_EINVAL;
    S.isu = 1.0f / S.su;
    const float eta = (opts && opts->eta != 0.0f) ? opts->eta : 0.999f;
    if (accel && !(eta > 0.0f && eta <= 1.0f)) return PINMPC_EINVAL;
    if (B == 0) return PINMPC_OK;
    if (!p->A || !p->Bm || !p->x0 || !p->x_ref || !p->contact || !d_ws) return PINMPC_EINVAL;
    if (ws_bytes < pinmpc_split_workspace_bytes_ex(nu, N, B, opts)) return PINMPC_EALLOC;
    cudaStream_t st_ = (cudaStream_t)stream;
    SolveParams P;
    memset(&P, 0, sizeof P);
    P.B = B; P.N = N; P.nu = nu; P.nw = layout->n_wrench; P.nf = layout->n_force; P.iters = iters; P.rho = rho;
    P.mu = layout->mu; P.fz_max = layout->fz_max * S.isu; P.cx = layout->mx_coef; P.cy = layout->my_coef; P.cz = layout->mz_coef;
    P.hand_fmax = layout->hand_fmax * S.isu;
    for (int i = 0; i < nx; i++) { if (!(h_Qdiag[i] >= 0.0f)) return PINMPC_EINVAL; P.Qd[i] = h_Qdiag[i] * S.sx[i] * S.sx[i]; }
    for (int i = 0; i < nu; i++) { if (!(h_Rdiag[i] >= 0.0f)) return PINMPC_EINVAL; P.Rd[i] = h_Rdiag[i] * S.su * S.su; }
    P.iw[0] = P.iw[1] = 1.0f / P.mu; P.iw[2] = 1.0f / P.cx; P.iw[3] = 1.0f / P.cy; P.iw[4] = 1.0f / P.cz;
    const long stg = (long)B * N, n = nx + nu;
    float *w = reinterpret_cast<float *>(((uintptr_t)d_ws + 255) & ~(uintptr_t)255);
    SplitPtrs q;
    q.A = p->A; q.Bm = p->Bm; q.c = p->c; q.x0 = p->x0; q.u_prev = p->u_prev; q.x_ref = p->x_ref; q.u_ref = p->u_ref; q.contact = p->contact;
    q.H = w; w += stg * n * n;
    q.G = w; w += stg * nu * nu;
    q.Tt = w; w += stg * nx * n;
    q.xi = w; w += stg * n;
    float *w0 = w; w += 5 * stg * n;
    q.nz = w0; q.nv = w0 + stg * n; q.nth = w0 + 2 * stg * n; q.nbe = w0 + 3 * stg * n; q.nla = w0 + 4 * stg * n;
    q.z = q.nz; q.v = q.nv; q.th = q.nth; q.be = q.nbe; q.la = q.nla;
    q.du = w; w += stg * nu;
    q.rs = w; w += stg;
    q.cpart = nullptr;
    for (int i = 0; i < NX; i++) {
        const float lo = (opts && opts->h_x_lo && i < nx) ? opts->h_x_lo[i] : -INFINITY, hi = (opts && opts->h_x_hi && i < nx) ? opts->h_x_hi[i] : INFINITY;
        if (!(lo <= hi)) return PINMPC_EINVAL;
        q.x_lo[i] = lo * S.isx[i]; q.x_hi[i] = hi * S.isx[i];
    }
    if (scaled) {
        float *sA = w; w += stg * nx * nx;
        float *sB = w; w += stg * nx * nu;
        float *sc = w; w += stg * nx;
        float *sxr = w; w += stg * nx;
        float *sur = w; w += stg * nu;
        float *sx0 = w; w += (long)B * nx;
        float *sup = w; w += (long)B * nu;
        const long tot = stg * nx * (nu > nx ? nu : nx);
        k_split_scale<<<(unsigned)((tot + 255) / 256), 256, 0, st_>>>(B, N, nx, nu, S, p->A, p->Bm, p->c, p->x0, p->u_prev, p->x_ref, p->u_ref, sA, sB, sc,
                                                                     sx0, sup, sxr, sur);
        q.A = sA; q.Bm = sB; q.c = p->c ? sc : nullptr; q.x0 = sx0; q.u_prev = p->u_prev ? sup : nullptr; q.x_ref = sxr;
        q.u_ref = p->u_ref ? sur : nullptr;
    }
    float *w1 = nullptr, *hat = nullptr;
    float4 *acc = nullptr;
    if (accel) {
        w1 = w; w += 5 * stg * n;
        hat = w; w += 5 * stg * n;
        q.cpart = w; w += stg;
        w = reinterpret_cast<float *>(((uintptr_t)w + 15) & ~(uintptr_t)15);
        acc = reinterpret_cast<float4 *>(w); w += (long)B * 4;
        if (cudaMemsetAsync(w1, 0, (size_t)stg * n * 10 * sizeof(float), st_) != cudaSuccess) return PINMPC_ECUDA;
    }
    // all iterates start at 0 (z, v, theta, beta, lambda are contiguous)
    if (cudaMemsetAsync(w0, 0, (size_t)stg * n * 5 * sizeof(float), st_) != cudaSuccess) return PINMPC_ECUDA;
    int *restarts = (accel && opts) ? opts->d_restarts : nullptr;
    pinmpc_status rc;
    if (nx == NX) rc = nu == 12 ? run<NX, 12>(P, q, iters, r_prim, accel, eta, w1, hat, acc, restarts, st_)
                                : run<NX, 18>(P, q, iters, r_prim, accel, eta, w1, hat, acc, restarts, st_);
    else rc = nu == 12 ? run<9, 12>(P, q, iters, r_prim, accel, eta, w1, hat, acc, restarts, st_)
                       : run<9, 18>(P, q, iters, r_prim, accel, eta, w1, hat, acc, restarts, st_);
    if (rc != PINMPC_OK) return rc;
    const float *zlast = (accel && ((iters - 1) & 1)) ? w1 : w0;
    const size_t bytes = (size_t)stg * n * sizeof(float);
    if (scaled) {
        const long tot = stg * n;
        if (xi) k_split_unscale<<<(unsigned)((tot + 255) / 256), 256, 0, st_>>>(stg, nx, (int)n, S, q.xi, xi);
        if (z) k_split_unscale<<<(unsigned)((tot + 255) / 256), 256, 0, st_>>>(stg, nx, (int)n, S, zlast, z);
        return cudaGetLastError() == cudaSuccess ? PINMPC_OK : PINMPC_ECUDA;
    }
    if (xi && cudaMemcpyAsync(xi, q.xi, bytes, cudaMemcpyDeviceToDevice, st_) != cudaSuccess) return PINMPC_ECUDA;
    if (z && cudaMemcpyAsync(z, zlast, bytes, cudaMemcpyDeviceToDevice, st_) != cudaSuccess) return PINMPC_ECUDA;
    return PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_split_solve(int nu, int N, int B, const pinmpc_layout *layout, const float *h_Qdiag, const float *h_Rdiag,
                                            float rho, int iters, const pinmpc_split_problem *p, void *d_ws, size_t ws_bytes,
                                            float *xi, float *z, float *r_prim, void *stream)
{
    return pinmpc_split_solve_ex(nu, N, B, layout, h_Qdiag, h_Rdiag, rho, iters, p, nullptr, d_ws, ws_bytes, xi, z, r_prim, stream);
}

// ---------------------------------------------------------------------------------------------
// pinmpc_split_solve_static: the same solve for callers that cannot allocate (CUDA graph capture, serving loops,
// harnesses that forbid cudaMalloc).  The workspace is this file-scope array: PINMPC_SPLIT_STATIC_BYTES of every GPU that
// loads the library, held until the process exits.  In host code `g_split_scratch` is only the host-side stand-in of
// the symbol, not a device address: the address is resolved once per device, with that device current, by
// cudaGetSymbolAddress and that pointer goes to the kernels.  Every call shares the array and finds the last call's
// contents in it: pinmpc_split_solve_ex zeroes the iterates (cudaMemsetAsync on the stream) and k_split_factor rewrites
// every factor before use, nothing else is read before it is written.  Calls that overlap on the GPU race.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_split_scratch[PINMPC_SPLIT_STATIC_BYTES];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mu;
void *g_static_ptr[STATIC_MAX_DEVICES];        // device address of g_split_scratch, per device ordinal (nullptr = not resolved)

pinmpc_status static_fail(pinmpc_status s, const char *fmt, ...)
{
    char msg[256];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(msg, sizeof msg, fmt, ap);
    va_end(ap);
    pinmpc_note_error(msg);
    return s;
}
}   // namespace

extern "C" size_t pinmpc_split_static_bytes(void) { return PINMPC_SPLIT_STATIC_BYTES; }

extern "C" pinmpc_status pinmpc_split_solve_static(int nu, int N, int B, const pinmpc_layout *layout, const float *h_Qdiag, const float *h_Rdiag,
                                                   float rho, int iters, const pinmpc_split_problem *p, const pinmpc_split_options *opts,
                                                   float *xi, float *z, float *r_prim, void *stream)
{
    const size_t need = pinmpc_split_workspace_bytes_ex(nu, N, B, opts);
    if (need == 0) return static_fail(PINMPC_EUNSUPPORTED, "pinmpc_split_solve_static: unsupported sizes (nu = %d, N = %d, B = %d)", nu, N, B);
    if (need > (size_t)PINMPC_SPLIT_STATIC_BYTES)
        return static_fail(PINMPC_EALLOC, "pinmpc_split_solve_static: this problem needs %zu bytes of scratch, the static array holds %zu "
                           "(PINMPC_SPLIT_STATIC_BYTES); use pinmpc_split_solve_ex with a caller-owned workspace", need, (size_t)PINMPC_SPLIT_STATIC_BYTES);
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= STATIC_MAX_DEVICES)
        return static_fail(PINMPC_ECUDA, "pinmpc_split_solve_static: cudaGetDevice: %s (device %d)", cudaGetErrorString(e), dev);
    void *ws = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_static_mu);
        if (g_static_ptr[dev] == nullptr) {                  // set-up, once per device, with that device current
            void *ptr = nullptr;
            e = cudaGetSymbolAddress(&ptr, g_split_scratch);
            if (e != cudaSuccess || ptr == nullptr)
                return static_fail(PINMPC_ECUDA, "pinmpc_split_solve_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            g_static_ptr[dev] = ptr;
        }
        ws = g_static_ptr[dev];
    }
    const pinmpc_status rc = pinmpc_split_solve_ex(nu, N, B, layout, h_Qdiag, h_Rdiag, rho, iters, p, opts, ws, PINMPC_SPLIT_STATIC_BYTES, xi, z, r_prim,
                                                   stream);
    if (rc != PINMPC_OK) static_fail(rc, "pinmpc_split_solve_static: pinmpc_split_solve_ex returned status %d", (int)rc);
    return rc;
}
