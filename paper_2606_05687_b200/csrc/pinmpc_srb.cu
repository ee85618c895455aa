// pinmpc_srb.cu — the STRUCTURED on-chip solver (PINMPC_METHOD_SRB), the product path.
//
// A_k and B_k are never formed ("construction-free"): the single-rigid-body
// structure of BASELINE.json config 0 (SRB form of PAPER.md eq. (2)-(4))
//     A_k = I + dt [Theta <- R_z^T omega, p <- v, v_z <- g],     B_k = E Bh_k,
//     E = rows 6..11 (omega, v),   Bh_k = D_k Gh_k,   D_k = blkdiag(dt I_w^-1, dt/m I),
//     Gh_k u = (sum_i r_i x f_i + sum_i m_i ;  sum_i f_i)          (net wrench about the CoM)
// lets the equality-constrained step (21a) be solved EXACTLY as an LQR in the 6-D input
// w = Bh_k u (the momentum increment) instead of the nu-D input u:
//   for given w the best u is  u = u0 + Rt^-1 Gh^T Lam^-1 (D^-1 w - Gh u0),  u0 = Rt^-1 r,
//   Lam = Gh Rt^-1 Gh^T, and its cost is 1/2 (w - w0)^T S (w - w0) + const, S = D^-1 Lam^-1 D^-1,
//   so with P_N = Q, for k = N-1..0
//     Mh = S_k + E^T P E,  Kh = Mh^-1 E^T P A_k (6x13),  P <- [k>=1] Q + A^T P A - G^T Kh,  G = E^T P A
//   backward  g = p - s;  hh = S w0 + E^T g;  p <- q + A^T g - Kh^T hh;   kappa = Mh^-1 hh
//   forward   w = kappa - Kh x;  x+ = A x + E (w + ch)
// The value function P_k and the iterates (x,u) equal those of the dense recursion of SURVEY.md
// 8(c)-O2/O3 (the oracle) up to rounding.
//
// Three kernels per solve:
//   k_assemble_srb  S1   one thread per (env, stage): geometry, Lam^-1, S, R ubar, Q xbar, ch
//   k_factor_srb    S2   one warp per env: the 13-state Riccati recursion in the 6-D input
//   k_iterate_srb   S3-6 one CTA per G envs, all ADMM iterations with every factor on chip:
//                        Kh and the exchange vectors in shared memory, the per-stage symmetric blocks,
//                        z and y in the registers of the thread that owns the stage (lane = stage);
//                        the two sequential passes run in warp 0, 8 lanes per env.
#include "pinmpc_common.cuh"

namespace {

constexpr int NW = 2;   // 6-D wrench contacts (feet)
constexpr unsigned FULL = 0xffffffffu;

__host__ __device__ constexpr int sidx(int i, int j)   // packed upper triangle of a symmetric 6x6
{
    return i <= j ? (i * 6 - i * (i - 1) / 2 + (j - i)) : (j * 6 - j * (j - 1) / 2 + (i - j));
}

__device__ __forceinline__ int fcol(int i) { return i < NW ? 3 * i : 6 * NW + 3 * (i - NW); }
__device__ __forceinline__ int mcol(int i) { return 3 * NW + 3 * i; }

// y = M x for packed symmetric 6x6 held in registers
__device__ __forceinline__ void symv6(const float *M, const float *x, float *y)
{
#pragma unroll
    for (int i = 0; i < 6; i++) {
        float a = 0.0f;
#pragma unroll
        for (int j = 0; j < 6; j++) a = fmaf(M[sidx(i, j)], x[j], a);
        y[i] = a;
    }
}

// In-place inverse of a packed symmetric positive definite 6x6 (Cholesky, registers of one thread).
__device__ __forceinline__ void spd_inv6(float *Mp)
{
    float L[6][6], Li[6][6];
#pragma unroll
    for (int j = 0; j < 6; j++) {
        float d = Mp[sidx(j, j)];
#pragma unroll
        for (int l = 0; l < j; l++) d = fmaf(-L[j][l], L[j][l], d);
        float dj = sqrtf(d), idj = 1.0f / dj;
        L[j][j] = dj;
#pragma unroll
        for (int i = j + 1; i < 6; i++) {
            float a = Mp[sidx(i, j)];
#pragma unroll
            for (int l = 0; l < j; l++) a = fmaf(-L[i][l], L[j][l], a);
            L[i][j] = a * idj;
        }
    }
#pragma unroll
    for (int c = 0; c < 6; c++) {
        Li[c][c] = 1.0f / L[c][c];
#pragma unroll
        for (int i = c + 1; i < 6; i++) {
            float a = 0.0f;
#pragma unroll
            for (int l = c; l < i; l++) a = fmaf(-L[i][l], Li[l][c], a);
            Li[i][c] = a / L[i][i];
        }
    }
#pragma unroll
    for (int i = 0; i < 6; i++)
#pragma unroll
        for (int j = i; j < 6; j++) {
            float a = 0.0f;
#pragma unroll
            for (int l = j; l < 6; l++) a = fmaf(Li[l][i], Li[l][j], a);
            Mp[sidx(i, j)] = a;
        }
}

// D^-1 v = (I_w v_tau / dt ; m v_F / dt) with I_w packed symmetric 3x3 (xx,xy,xz,yy,yz,zz)
__device__ __forceinline__ void dinv_apply(const float *Iw, float idt, float m_dt, const float *v, float *o)
{
    o[0] = (Iw[0] * v[0] + Iw[1] * v[1] + Iw[2] * v[2]) * idt;
    o[1] = (Iw[1] * v[0] + Iw[3] * v[1] + Iw[4] * v[2]) * idt;
    o[2] = (Iw[2] * v[0] + Iw[4] * v[1] + Iw[5] * v[2]) * idt;
    o[3] = v[3] * m_dt; o[4] = v[4] * m_dt; o[5] = v[5] * m_dt;
}

// u0 = Rt^-1 (R ubar + rho (z - y)) and its net wrench G0 = Gh u0 for one stage (thread-local)
template <int NU>
__device__ __forceinline__ void stage_u0(const SolveParams &P, const float *ru, const float *z, const float *y,
                                         const float *r, float *u0, float *G0)
{
    constexpr int NC = NW + (NU - 12) / 3;
#pragma unroll
    for (int j = 0; j < NU; j++) u0[j] = (ru[j] + P.rho * (z[j] - y[j])) / (P.Rd[j] + P.rho);
#pragma unroll
    for (int a = 0; a < 6; a++) G0[a] = 0.0f;
#pragma unroll
    for (int i = 0; i < NC; i++) {
        const float *f = u0 + fcol(i);
        float rx = r[3 * i], ry = r[3 * i + 1], rz = r[3 * i + 2];
        G0[0] += ry * f[2] - rz * f[1];
        G0[1] += rz * f[0] - rx * f[2];
        G0[2] += rx * f[1] - ry * f[0];
        G0[3] += f[0]; G0[4] += f[1]; G0[5] += f[2];
        if (i < NW) {
            const float *m = u0 + mcol(i);
            G0[0] += m[0]; G0[1] += m[1]; G0[2] += m[2];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// S1  construction-free assembly: one thread per (env, stage)
// ---------------------------------------------------------------------------------------------
template <int NU>
__global__ void __launch_bounds__(128) k_assemble_srb(SolveParams P, ProblemPtrs q, SrbWs W)
{
    constexpr int NC = NW + (NU - 12) / 3;
    const long st = (long)P.B * P.N;
    const long s = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= st) return;
    const int N = P.N;
    const int b = (int)(s / N), k = (int)(s - (long)b * N);
    const float dt = P.dt, idt = 1.0f / P.dt;
    const float mass = q.mass[b], dtm = dt / mass, m_dt = mass / dt;

    float Ib[9];
#pragma unroll
    for (int i = 0; i < 9; i++) Ib[i] = q.inertia[(long)b * 9 + i];
    float sn, cs;
    sincosf(q.yaw[s], &sn, &cs);
    W.cs[s * 2] = cs; W.cs[s * 2 + 1] = sn;
    // I_w = R_z I_b R_z^T (same congruence as world_inertia_inv, applied to I_b)
    float Iwf[9];
    world_inertia_inv(Ib, cs, sn, Iwf);
    const float iw[6] = { Iwf[0], Iwf[1], Iwf[2], Iwf[4], Iwf[5], Iwf[8] };
#pragma unroll
    for (int i = 0; i < 6; i++) W.IW[i * st + s] = iw[i];

    int bits = 0;
    float r[3 * NC];
#pragma unroll
    for (int i = 0; i < NC; i++) {
        bits |= (q.contact[s * NC + i] != 0) << i;
#pragma unroll
        for (int a = 0; a < 3; a++) {
            r[3 * i + a] = q.foot_r[(s * NC + i) * 3 + a];
            W.RR[(3 * i + a) * st + s] = r[3 * i + a];
        }
    }
    W.bits[s] = bits;
#pragma unroll
    for (int j = 0; j < NU; j++) W.RU[j * st + s] = q.u_ref ? P.Rd[j] * q.u_ref[s * NU + j] : 0.0f;
    // q_{k+1} = Q xbar_{k+1}  (x_ref[b,k] holds xbar_{k+1});  q_0 = 0
    {
        float *qv = W.qv + ((long)b * (N + 1) + k + 1) * 12;
#pragma unroll
        for (int j = 0; j < 12; j++) qv[j] = P.Qd[j] * q.x_ref[s * NX + j];
        if (k == 0) {
            float *q0 = W.qv + (long)b * (N + 1) * 12;
#pragma unroll
            for (int j = 0; j < 12; j++) q0[j] = 0.0f;
        }
    }
    // Lam = Gh Rt^-1 Gh^T, accumulated column by column of Gh
    float Lam[21];
#pragma unroll
    for (int i = 0; i < 21; i++) Lam[i] = 0.0f;
#pragma unroll
    for (int i = 0; i < NC; i++) {
        float rx = r[3 * i], ry = r[3 * i + 1], rz = r[3 * i + 2];
        const float col[3][3] = { { 0.0f, rz, -ry }, { -rz, 0.0f, rx }, { ry, -rx, 0.0f } };   // r x e_a
#pragma unroll
        for (int a = 0; a < 3; a++) {
            float w = 1.0f / (P.Rd[fcol(i) + a] + P.rho);
            float g6[6] = { col[a][0], col[a][1], col[a][2], a == 0 ? 1.0f : 0.0f, a == 1 ? 1.0f : 0.0f, a == 2 ? 1.0f : 0.0f };
#pragma unroll
            for (int x = 0; x < 6; x++)
#pragma unroll
                for (int y = x; y < 6; y++) Lam[sidx(x, y)] = fmaf(w * g6[x], g6[y], Lam[sidx(x, y)]);
            if (i < NW) Lam[sidx(a, a)] += 1.0f / (P.Rd[mcol(i) + a] + P.rho);
        }
    }
    spd_inv6(Lam);                                   // Lam^-1
#pragma unroll
    for (int i = 0; i < 21; i++) W.LI[i * st + s] = Lam[i];
    // S = D^-1 Lam^-1 D^-1,  D^-1 = blkdiag(I_w / dt, m/dt I)
    {
        const float Iw3[3][3] = { { iw[0], iw[1], iw[2] }, { iw[1], iw[3], iw[4] }, { iw[2], iw[4], iw[5] } };
        float T[3][3], S[21];
#pragma unroll
        for (int x = 0; x < 3; x++)
#pragma unroll
            for (int y = 0; y < 3; y++) {
                float a = 0.0f;
#pragma unroll
                for (int l = 0; l < 3; l++) a = fmaf(Iw3[x][l], Lam[sidx(l, y)], a);
                T[x][y] = a;
            }
#pragma unroll
        for (int x = 0; x < 3; x++)
#pragma unroll
            for (int y = x; y < 3; y++) {
                float a = 0.0f;
#pragma unroll
                for (int l = 0; l < 3; l++) a = fmaf(T[x][l], Iw3[l][y], a);
                S[sidx(x, y)] = a * idt * idt;
            }
#pragma unroll
        for (int x = 0; x < 3; x++)
#pragma unroll
            for (int y = 0; y < 3; y++) {
                float a = 0.0f;
#pragma unroll
                for (int l = 0; l < 3; l++) a = fmaf(Iw3[x][l], Lam[sidx(l, 3 + y)], a);
                S[sidx(x, 3 + y)] = a * idt * m_dt;
            }
#pragma unroll
        for (int x = 0; x < 3; x++)
#pragma unroll
            for (int y = x; y < 3; y++) S[sidx(3 + x, 3 + y)] = Lam[sidx(3 + x, 3 + y)] * m_dt * m_dt;
#pragma unroll
        for (int i = 0; i < 21; i++) W.MI[i * st + s] = S[i];
    }
    // ch = (dt I_w^-1 tau_ext ; dt/m F_ext): the part of c_k in rows 6..11
    if (q.ext != nullptr) {
        float Ibi[9], Wi[9];
        inv3f(Ib, Ibi);
        world_inertia_inv(Ibi, cs, sn, Wi);
        const float *e = q.ext + s * 6;
#pragma unroll
        for (int a = 0; a < 3; a++) {
            W.c6[s * 6 + a] = dt * (Wi[a * 3] * e[3] + Wi[a * 3 + 1] * e[4] + Wi[a * 3 + 2] * e[5]);
            W.c6[s * 6 + 3 + a] = dtm * e[a];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// S2  factorisation: one warp per env, sequential over stages, P (13x13) in shared memory
// ---------------------------------------------------------------------------------------------
constexpr int FAC_WARPS = 4;                     // warps (envs) per CTA
constexpr int FAC_SMEM = 172 + 172 + 80 + 24;    // floats per warp: P, X, Kh, Mh^-1

// element (i,j) of A^T X for the structured A (rows 6..12 of A^T pick up dt * rows of X)
__device__ __forceinline__ float atx(const float *X, int i, int j, float dt, float cs, float sn)
{
    float a = X[i * NX + j];
    if (i == 6) a += dt * (cs * X[0 * NX + j] - sn * X[1 * NX + j]);
    else if (i == 7) a += dt * (sn * X[0 * NX + j] + cs * X[1 * NX + j]);
    else if (i == 8) a += dt * X[2 * NX + j];
    else if (i >= 9 && i <= 11) a += dt * X[(i - 6) * NX + j];
    else if (i == 12) a += dt * X[11 * NX + j];
    return a;
}

__global__ void __launch_bounds__(FAC_WARPS * 32) k_factor_srb(SolveParams P, const float *__restrict__ x0, SrbWs W, int has_ext)
{
    __shared__ __align__(16) float sm_all[FAC_WARPS * FAC_SMEM];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int b = blockIdx.x * FAC_WARPS + wib;
    if (b >= P.B) return;
    float *sP = sm_all + wib * FAC_SMEM, *sX = sP + 172, *sK = sX + 172, *sM = sK + 80;
    const int N = P.N;
    const long st = (long)P.B * N;
    const float dt = P.dt;
    const float x12 = x0[(long)b * NX + 12];

    // lane <-> (i,j) of the packed symmetric 6x6 (lanes >= 21 shadow element (0,0))
    int mi = 0, mj = 0;
    {
        int l = lane < 21 ? lane : 0, row = 0;
        while (l >= 6 - row) { l -= 6 - row; row++; }
        mi = row; mj = row + l;
    }
    int la[6], lb[6];
#pragma unroll
    for (int p = 0; p < 6; p++) { la[p] = sidx(mi, p); lb[p] = sidx(p, mj); }
    // upper triangle of the 13x13: element t = lane + 32 r  ->  (ti, tj), ti <= tj
    int ti[3], tj[3];
#pragma unroll
    for (int r = 0; r < 3; r++) {
        int t = lane + 32 * r, row = 0;
        if (t > 90) t = 90;
        while (t >= NX - row) { t -= NX - row; row++; }
        ti[r] = row; tj[r] = row + t;
    }

    for (int i = lane; i < 169; i += 32) sP[i] = ((i * 79) >> 10) * 14 == i ? P.Qd[(i * 79) >> 10] : 0.0f;
    __syncwarp();

    // prefetch stage N-1
    long s = (long)b * N + N - 1;
    float cs_n = W.cs[s * 2], sn_n = W.cs[s * 2 + 1];
    float S_n = W.MI[(long)(lane < 21 ? lane : 0) * st + s];
    float ch_n = (has_ext && lane < 6) ? W.c6[s * 6 + lane] : 0.0f;
    for (int k = N - 1; k >= 0; k--) {
        s = (long)b * N + k;
        const float cs = cs_n, sn = sn_n, Sl = S_n, chl = ch_n;
        if (k > 0) {
            cs_n = W.cs[(s - 1) * 2]; sn_n = W.cs[(s - 1) * 2 + 1];
            S_n = W.MI[(long)(lane < 21 ? lane : 0) * st + s - 1];
            ch_n = (has_ext && lane < 6) ? W.c6[(s - 1) * 6 + lane] : 0.0f;
        }
        // X = P A
#pragma unroll
        for (int r = 0; r < 6; r++) {
            int e = lane + 32 * r;
            if (e < 169) {
                int i = (e * 79) >> 10, j = e - i * NX;
                const float *Pi = sP + i * NX;
                float a = Pi[j];
                if (j == 6) a += dt * (cs * Pi[0] - sn * Pi[1]);
                else if (j == 7) a += dt * (sn * Pi[0] + cs * Pi[1]);
                else if (j == 8) a += dt * Pi[2];
                else if (j >= 9 && j <= 11) a += dt * Pi[j - 6];
                else if (j == 12) a += dt * Pi[11];
                sX[e] = a;
            }
        }
        // Mh = S + P[6:12,6:12] (one packed element per lane) ; s_k = P (E ch)
        float M = Sl + sP[(6 + mi) * NX + 6 + mj];
        float sk = 0.0f;
        if (has_ext) {
            const int rl = lane < NX ? lane : 0;
#pragma unroll
            for (int a = 0; a < 6; a++) sk = fmaf(sP[rl * NX + 6 + a], __shfl_sync(FULL, chl, a), sk);
        }
        // Mh^-1 by symmetric sweeps (-Mh^-1 after six pivots), all in registers
#pragma unroll
        for (int p = 0; p < 6; p++) {
            float d = __shfl_sync(FULL, M, sidx(p, p));
            float a = __shfl_sync(FULL, M, la[p]);
            float c = __shfl_sync(FULL, M, lb[p]);
            float id = 1.0f / d;
            if (mi == p && mj == p) M = -id;
            else if (mi == p || mj == p) M = M * id;
            else M = fmaf(-a * id, c, M);
        }
        M = -M;
        if (lane < 21) { sM[lane] = M; W.MI[(long)lane * st + s] = M; }
        __syncwarp();
        // Kh = Mh^-1 X[6:12,:]
#pragma unroll
        for (int r = 0; r < 3; r++) {
            int e = lane + 32 * r;
            if (e < 78) {
                int i = (e * 79) >> 10, j = e - i * NX;
                float a = 0.0f;
#pragma unroll
                for (int l = 0; l < 6; l++) a = fmaf(sM[sidx(i, l)], sX[(6 + l) * NX + j], a);
                sK[e] = a;
                if (j < 12) W.Kh[s * 72 + i * 12 + j] = a;
                else W.KG[(long)i * st + s] = a * x12;
            }
        }
        if (has_ext && lane < 12) W.sv[s * 12 + lane] = sk;
        __syncwarp();
        // P <- [k>=1] Q + A^T X - G^T Kh   (upper triangle, mirrored: both terms are symmetric)
#pragma unroll
        for (int r = 0; r < 3; r++) {
            if (lane + 32 * r < 91) {
                int i = ti[r], j = tj[r];
                float a = atx(sX, i, j, dt, cs, sn);
#pragma unroll
                for (int l = 0; l < 6; l++) a = fmaf(-sX[(6 + l) * NX + i], sK[l * NX + j], a);
                if (k >= 1 && i == j) a += P.Qd[i];
                sP[i * NX + j] = a;
                sP[j * NX + i] = a;
            }
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------
// S3-S6  ADMM iterations: one CTA per G envs, every factor on chip
// ---------------------------------------------------------------------------------------------
// Shared-memory arena of one env (offsets in floats).  The arena stride is 8 mod 32 so that the
// 8-lane groups of up to four envs in the pass warp hit disjoint banks.
struct ArenaLay { int oQ, oX, oCS, oM, oC, oS, oF, stride; };

__host__ __device__ inline ArenaLay arena_layout(int N, int ext)
{
    ArenaLay L;
    L.oQ = 72 * N;                    // Kh [N][6][12] at 0 ; q [N+1][12]
    L.oX = L.oQ + 12 * (N + 1);       // exchange vector [N][8]: sigma0 -> hh -> kappa -> w
    L.oCS = L.oX + 8 * N;             // cos, sin [N][2]
    L.oM = L.oCS + 2 * N;             // Mh^-1 (21) and kg (6) per stage, stride 27 (lane = stage)
    L.oC = L.oM + 27 * N;             // ch [N][6]      (ext only)
    L.oS = L.oC + (ext ? 6 * N : 0);  // s  [N][12]     (ext only)
    L.oF = (L.oS + (ext ? 12 * N : 0) + 3) & ~3;   // forward-pass exchange scratch [2][8]
    int size = L.oF + 16;
    L.stride = size + ((8 - (size & 31)) & 31);
    return L;
}

constexpr int CTL_INTS = 32;          // done[4] | ndone | pad[3] | red[4][5]

// Backward vector pass of all envs of the CTA (warp 0; lane = 8 e + i, lanes i < 6 own the
// columns i (Theta/p part) and 6 + i (omega/v part) of p).
__device__ __forceinline__ void backward_pass(const ArenaLay &L, float *smem, int N, int Gv, float dt, int has_ext, int lane)
{
    const int e = lane >> 3, i0 = lane & 7, i = i0 < 6 ? i0 : 5;
    const bool act = i0 < 6 && e < Gv;
    float *ar = smem + (e < Gv ? e : 0) * L.stride;
    const float *aQ = ar + L.oQ, *aCS = ar + L.oCS, *aS = ar + L.oS;
    float *aX = ar + L.oX;
    float pq = aQ[N * 12 + i], pv = aQ[N * 12 + 6 + i];
    for (int k = N - 1; k >= 0; k--) {
        const float *Kk = ar + k * 72;
        float kq[6], kv[6];
#pragma unroll
        for (int r = 0; r < 6; r++) { kq[r] = Kk[r * 12 + i]; kv[r] = Kk[r * 12 + 6 + i]; }
        const float qq = aQ[k * 12 + i], qn = aQ[k * 12 + 6 + i];
        const float s0 = aX[k * 8 + i];
        const float csk = aCS[2 * k], snk = aCS[2 * k + 1];
        float sq = 0.0f, sn6 = 0.0f;
        if (has_ext) { sq = aS[k * 12 + i]; sn6 = aS[k * 12 + 6 + i]; }
        const float gq = pq - sq, gv = pv - sn6;
        const float hh = s0 + gv;
        if (act) aX[k * 8 + i] = hh;
        const float oth = __shfl_xor_sync(FULL, gq, 1);
        __syncwarp();
        const float4 h0 = *reinterpret_cast<const float4 *>(aX + k * 8);
        const float2 h1 = *reinterpret_cast<const float2 *>(aX + k * 8 + 4);
        float a0 = kq[0] * h0.x, a1 = kq[3] * h0.w, b0 = kv[0] * h0.x, b1 = kv[3] * h0.w;
        a0 = fmaf(kq[1], h0.y, a0); a1 = fmaf(kq[4], h1.x, a1); b0 = fmaf(kv[1], h0.y, b0); b1 = fmaf(kv[4], h1.x, b1);
        a0 = fmaf(kq[2], h0.z, a0); a1 = fmaf(kq[5], h1.y, a1); b0 = fmaf(kv[2], h0.z, b0); b1 = fmaf(kv[5], h1.y, b1);
        // (A^T g)_nu = g_nu + dt (R_z g_Theta ; g_p)
        const float ca = i < 2 ? csk : 1.0f, cb = i == 0 ? -snk : (i == 1 ? snk : 0.0f);
        const float rot = fmaf(cb, oth, ca * gq);
        pq = (qq + gq) - (a0 + a1);
        pv = fmaf(dt, rot, qn + gv) - (b0 + b1);
    }
}

// Forward rollout of all envs of the CTA (warp 0; every active lane holds the whole state, lane i
// owns row i of Kh and the new omega/v component i).  Writes w_k over kappa_k; optionally emits x.
__device__ __forceinline__ void forward_pass(const ArenaLay &L, float *smem, int N, int Gv, float dt, int has_ext, int lane,
                                             const float *__restrict__ x0g, int b0, bool emit, const int *done, float *ox)
{
    const int e = lane >> 3, i0 = lane & 7, i = i0 < 6 ? i0 : 5;
    const bool act = i0 < 6 && e < Gv;
    const int ee = e < Gv ? e : 0;
    float *ar = smem + ee * L.stride;
    const float *aCS = ar + L.oCS, *aC = ar + L.oC;
    float *aX = ar + L.oX, *aF = ar + L.oF;
    const float *xg = x0g + (long)(b0 + ee) * NX;
    float x0 = xg[0], x1 = xg[1], x2 = xg[2], x3 = xg[3], x4 = xg[4], x5 = xg[5];
    float x6 = xg[6], x7 = xg[7], x8 = xg[8], x9 = xg[9], x10 = xg[10], x11 = xg[11];
    const float x12 = xg[12];
    float own = xg[6 + i];
    const float gdt = i == 5 ? dt * x12 : 0.0f;
    const bool wr = emit && act && !done[ee];
    float *oxe = ox + (long)(b0 + ee) * N * NX;
    int par = 0;
    for (int k = 0; k < N; k++) {
        const float4 *Kr = reinterpret_cast<const float4 *>(ar + k * 72 + i * 12);
        const float4 r0 = Kr[0], r1 = Kr[1], r2 = Kr[2];
        const float kap = aX[k * 8 + i];
        const float csk = aCS[2 * k], snk = aCS[2 * k + 1];
        const float c = (has_ext ? aC[k * 6 + i] : 0.0f) + gdt;
        float a0 = r0.x * x0, a1 = r0.w * x3, a2 = r1.z * x6, a3 = r2.y * x9;
        a0 = fmaf(r0.y, x1, a0); a1 = fmaf(r1.x, x4, a1); a2 = fmaf(r1.w, x7, a2); a3 = fmaf(r2.z, x10, a3);
        a0 = fmaf(r0.z, x2, a0); a1 = fmaf(r1.y, x5, a1); a2 = fmaf(r2.x, x8, a2); a3 = fmaf(r2.w, x11, a3);
        const float w = kap - ((a0 + a1) + (a2 + a3));
        const float nun = own + (w + c);
        if (act) { aX[k * 8 + i] = w; aF[par * 8 + i] = nun; }
        // Theta+ = Theta + dt R_z^T omega ; p+ = p + dt v   (old omega, v)
        x0 = fmaf(dt, fmaf(csk, x6, snk * x7), x0);
        x1 = fmaf(dt, fmaf(csk, x7, -snk * x6), x1);
        x2 = fmaf(dt, x8, x2); x3 = fmaf(dt, x9, x3); x4 = fmaf(dt, x10, x4); x5 = fmaf(dt, x11, x5);
        __syncwarp();
        const float4 n0 = *reinterpret_cast<const float4 *>(aF + par * 8);
        const float2 n1 = *reinterpret_cast<const float2 *>(aF + par * 8 + 4);
        x6 = n0.x; x7 = n0.y; x8 = n0.z; x9 = n0.w; x10 = n1.x; x11 = n1.y;
        own = nun;
        if (wr) {
            const float xs = i == 0 ? x0 : i == 1 ? x1 : i == 2 ? x2 : i == 3 ? x3 : i == 4 ? x4 : x5;
            oxe[k * NX + i] = xs;
            oxe[k * NX + 6 + i] = nun;
            if (i == 0) oxe[k * NX + 12] = x12;
        }
        par ^= 1;
    }
}

template <int NU>
__global__ void __launch_bounds__(256) k_iterate_srb(SolveParams P, SrbWs W, const float *__restrict__ x0g,
                                                     const float *__restrict__ massg, OutPtrs o, int G, int has_ext)
{
    constexpr int NC = NW + (NU - 12) / 3;
    extern __shared__ __align__(16) float smem[];
    const int N = P.N, tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const long st = (long)P.B * N;
    const ArenaLay L = arena_layout(N, has_ext);
    const int b0 = blockIdx.x * G;
    const int Gv = min(G, P.B - b0);
    int *ctl = reinterpret_cast<int *>(smem + G * L.stride);
    int *done = ctl, *ndone = ctl + 4;
    unsigned *red = reinterpret_cast<unsigned *>(ctl + 8);
    const float dt = P.dt, idt = 1.0f / P.dt;

    // this thread's stage task: env te of the CTA, stage tk
    const int te = tid / N, tk = tid - te * N;
    const bool tact = te < Gv;
    const int bb = b0 + (tact ? te : 0);
    const long ts = (long)bb * N + tk;
    float *ar = smem + (tact ? te : 0) * L.stride;
    float *myX = ar + L.oX + tk * 8, *myM = ar + L.oM + tk * 27;

    // ---- load the pass arrays of the CTA's envs into shared memory ------------------------------
    for (int e = 0; e < Gv; e++) {
        float *a = smem + e * L.stride;
        const long s0 = (long)(b0 + e) * N;
        const float4 *src = reinterpret_cast<const float4 *>(W.Kh + s0 * 72);
        float4 *dst = reinterpret_cast<float4 *>(a);
        for (int i = tid; i < N * 18; i += nthr) dst[i] = src[i];
        src = reinterpret_cast<const float4 *>(W.qv + (long)(b0 + e) * (N + 1) * 12);
        dst = reinterpret_cast<float4 *>(a + L.oQ);
        for (int i = tid; i < (N + 1) * 3; i += nthr) dst[i] = src[i];
        for (int i = tid; i < N * 2; i += nthr) a[L.oCS + i] = W.cs[s0 * 2 + i];
        if (has_ext) {
            for (int i = tid; i < N * 6; i += nthr) a[L.oC + i] = W.c6[s0 * 6 + i];
            for (int i = tid; i < N * 12; i += nthr) a[L.oS + i] = W.sv[s0 * 12 + i];
        }
    }
    if (tid < CTL_INTS) ctl[tid] = 0;

    // ---- stage-stationary registers (lane = stage) ---------------------------------------------
    float LI[21], Iw[6], r[3 * NC], ru[NU], z[NU], y[NU];
    int bits = 0;
    float m_dt = 0.0f;
    if (tact) {
#pragma unroll
        for (int c = 0; c < 21; c++) { LI[c] = W.LI[c * st + ts]; myM[c] = W.MI[c * st + ts]; }
#pragma unroll
        for (int c = 0; c < 6; c++) { Iw[c] = W.IW[c * st + ts]; myM[21 + c] = W.KG[c * st + ts]; }
#pragma unroll
        for (int c = 0; c < 3 * NC; c++) r[c] = W.RR[c * st + ts];
#pragma unroll
        for (int c = 0; c < NU; c++) { ru[c] = W.RU[c * st + ts]; z[c] = 0.0f; y[c] = 0.0f; }
        bits = W.bits[ts];
        m_dt = massg[bb] / dt;
    }

    // sigma0 = D^-1 Lam^-1 Gh u0 of the coming iteration from the current z, y  (phase P1)
    auto stage_sigma0 = [&]() {
        float u0[NU], G0[6], l0[6], s0[6];
        stage_u0<NU>(P, ru, z, y, r, u0, G0);
        symv6(LI, G0, l0);
        dinv_apply(Iw, idt, m_dt, l0, s0);
        *reinterpret_cast<float4 *>(myX) = make_float4(s0[0], s0[1], s0[2], s0[3]);
        *reinterpret_cast<float2 *>(myX + 4) = make_float2(s0[4], s0[5]);
    };
    if (tact) stage_sigma0();

    const bool tol_mode = (P.eps_abs > 0.0f || P.eps_rel > 0.0f) && P.check_every > 0;
    bool frozen = false;          // this thread's env has met the tolerances (tolerance mode only)

    for (int it = 0; it < P.iters; it++) {
        const bool is_check = tol_mode && ((it + 1) % P.check_every == 0);
        const bool emit = (it == P.iters - 1) || is_check;
        __syncthreads();                                   // sigma0 of every stage is in place
        if (warp == 0) backward_pass(L, smem, N, Gv, dt, has_ext, lane);
        __syncthreads();
        // ---- P2: kappa = Mh^-1 hh - Kh[:,12] x_12  (lane = stage) ----------------------------------
        if (tact) {
            const float4 h0 = *reinterpret_cast<const float4 *>(myX);
            const float2 h1 = *reinterpret_cast<const float2 *>(myX + 4);
            const float h[6] = { h0.x, h0.y, h0.z, h0.w, h1.x, h1.y };
            float Mi[21], kp[6];
#pragma unroll
            for (int c = 0; c < 21; c++) Mi[c] = myM[c];
            symv6(Mi, h, kp);
#pragma unroll
            for (int a = 0; a < 6; a++) kp[a] -= myM[21 + a];
            *reinterpret_cast<float4 *>(myX) = make_float4(kp[0], kp[1], kp[2], kp[3]);
            *reinterpret_cast<float2 *>(myX + 4) = make_float2(kp[4], kp[5]);
        }
        if (emit && tid < 20) red[tid] = 0u;
        __syncthreads();
        if (warp == 0) forward_pass(L, smem, N, Gv, dt, has_ext, lane, x0g, b0, emit, done, o.x);
        __syncthreads();
        // ---- P3: u from w, projection (S4), dual update (S5), residuals (S6)  (lane = stage) --------
        if (tact && !frozen) {
            float u0[NU], G0[6], wv[6], dl[6], lam[6];
            stage_u0<NU>(P, ru, z, y, r, u0, G0);
            {
                const float4 w0 = *reinterpret_cast<const float4 *>(myX);
                const float2 w1 = *reinterpret_cast<const float2 *>(myX + 4);
                wv[0] = w0.x; wv[1] = w0.y; wv[2] = w0.z; wv[3] = w0.w; wv[4] = w1.x; wv[5] = w1.y;
            }
            dinv_apply(Iw, idt, m_dt, wv, dl);
#pragma unroll
            for (int a = 0; a < 6; a++) dl[a] -= G0[a];
            symv6(LI, dl, lam);
            // u = u0 + Rt^-1 Gh^T lam :  f_i += lam_tau x r_i + lam_F ;  m_i += lam_tau
            float u[NU];
#pragma unroll
            for (int i = 0; i < NC; i++) {
                float rx = r[3 * i], ry = r[3 * i + 1], rz = r[3 * i + 2];
                float c0 = lam[1] * rz - lam[2] * ry + lam[3];
                float c1 = lam[2] * rx - lam[0] * rz + lam[4];
                float c2 = lam[0] * ry - lam[1] * rx + lam[5];
                const int fc = fcol(i);
                u[fc] = u0[fc] + c0 / (P.Rd[fc] + P.rho);
                u[fc + 1] = u0[fc + 1] + c1 / (P.Rd[fc + 1] + P.rho);
                u[fc + 2] = u0[fc + 2] + c2 / (P.Rd[fc + 2] + P.rho);
                if (i < NW) {
                    const int mc = mcol(i);
#pragma unroll
                    for (int a = 0; a < 3; a++) u[mc + a] = u0[mc + a] + lam[a] / (P.Rd[mc + a] + P.rho);
                }
            }
            float zn[NU];
#pragma unroll
            for (int i = 0; i < NC; i++) {
                const bool on = (bits >> i) & 1;
                const int fc = fcol(i);
                if (i < NW) {
                    const int mc = mcol(i);
                    float a0, a1, a2, a3, a4, a5;
                    project_wrench(P, u[fc] + y[fc], u[fc + 1] + y[fc + 1], u[fc + 2] + y[fc + 2], u[mc] + y[mc],
                                   u[mc + 1] + y[mc + 1], u[mc + 2] + y[mc + 2], a0, a1, a2, a3, a4, a5);
                    zn[fc] = on ? a0 : 0.0f; zn[fc + 1] = on ? a1 : 0.0f; zn[fc + 2] = on ? a2 : 0.0f;
                    zn[mc] = on ? a3 : 0.0f; zn[mc + 1] = on ? a4 : 0.0f; zn[mc + 2] = on ? a5 : 0.0f;
                } else {
#pragma unroll
                    for (int a = 0; a < 3; a++)
                        zn[fc + a] = on ? fminf(fmaxf(u[fc + a] + y[fc + a], -P.hand_fmax), P.hand_fmax) : 0.0f;
                }
            }
            if (emit) {
                float rp = 0.0f, rd = 0.0f, un = 0.0f, znm = 0.0f, ynm = 0.0f;
                float *ou = o.u + ts * NU;
#pragma unroll
                for (int j = 0; j < NU; j++) {
                    rp = fmaxf(rp, fabsf(u[j] - zn[j]));
                    rd = fmaxf(rd, fabsf(zn[j] - z[j]));
                    un = fmaxf(un, fabsf(u[j])); znm = fmaxf(znm, fabsf(zn[j]));
                    ynm = fmaxf(ynm, fabsf(y[j] + u[j] - zn[j]));
                    ou[j] = u[j];
                }
                // non-negative floats order like their bit patterns
                atomicMax(&red[te * 5 + 0], __float_as_uint(rp)); atomicMax(&red[te * 5 + 1], __float_as_uint(rd));
                atomicMax(&red[te * 5 + 2], __float_as_uint(un)); atomicMax(&red[te * 5 + 3], __float_as_uint(znm));
                atomicMax(&red[te * 5 + 4], __float_as_uint(ynm));
            }
#pragma unroll
            for (int j = 0; j < NU; j++) { y[j] = y[j] + u[j] - zn[j]; z[j] = zn[j]; }
        }
        if (emit) {
            __syncthreads();
            if (tid < Gv && !done[tid]) {                  // one leader per env
                const float rp = __uint_as_float(red[tid * 5 + 0]), rd = P.rho * __uint_as_float(red[tid * 5 + 1]);
                o.r_prim[b0 + tid] = rp; o.r_dual[b0 + tid] = rd; o.iters_done[b0 + tid] = it + 1;
                if (is_check) {
                    const float sc = fmaxf(__uint_as_float(red[tid * 5 + 2]), __uint_as_float(red[tid * 5 + 3]));
                    const float ys = __uint_as_float(red[tid * 5 + 4]);
                    if (rp <= P.eps_abs + P.eps_rel * sc && rd <= P.eps_abs + P.eps_rel * P.rho * ys) {
                        done[tid] = 1;
                        atomicAdd(ndone, 1);
                    }
                }
            }
            __syncthreads();
            if (is_check) {
                if (*ndone == Gv) break;
                if (tact) frozen = done[te] != 0;
            }
        }
        if (tact && it + 1 < P.iters) stage_sigma0();      // frozen envs keep a well-defined (constant) sigma0
    }
    if (tact) {
        float *oz = o.z + ts * NU, *oy = o.y + ts * NU;
#pragma unroll
        for (int j = 0; j < NU; j++) { oz[j] = z[j]; oy[j] = y[j]; }
    }
}

// ---------------------------------------------------------------------------------------------
// launcher
// ---------------------------------------------------------------------------------------------
int fail(pinmpc_ctx *h, const char *what, cudaError_t e)
{
    h->sticky = e;
    snprintf(h->err, sizeof h->err, "%s: %s", what, cudaGetErrorString(e));
    return -1;
}

size_t iterate_smem_bytes(int N, int G, int ext)
{
    return ((size_t)G * arena_layout(N, ext).stride + CTL_INTS) * sizeof(float);
}

// envs per CTA: the G in 1..4 that keeps most envs resident per SM (shared memory, registers and
// thread slots), ties to the smaller CTA (more independent CTAs overlap passes and stage phases).
int choose_G(const pinmpc_ctx *h, int regs, int ext)
{
    int best = 0, best_envs = 0;
    for (int G = 1; G <= 4; G++) {
        int threads = (G * h->N + 31) / 32 * 32;
        if (threads < 32) threads = 32;
        size_t smem = iterate_smem_bytes(h->N, G, ext);
        if (threads > 256 || smem > (size_t)h->smem_optin) continue;
        int by_smem = (int)((size_t)(228 * 1024) / (smem + 1024));
        int by_regs = 65536 / (threads * ((regs + 7) / 8 * 8));
        int by_thr = 2048 / threads;
        int ctas = by_smem < by_regs ? by_smem : by_regs;
        if (by_thr < ctas) ctas = by_thr;
        if (ctas > 32) ctas = 32;
        if (ctas < 1) continue;
        int envs = ctas * G;
        if (envs > best_envs) { best_envs = envs; best = G; }
    }
    return best;
}

template <int NU>
int launch_t(pinmpc_ctx *h, cudaStream_t st)
{
    SolveParams P = make_params(h);
    ProblemPtrs q = make_problem_ptrs(h);
    const int ext = q.ext != nullptr;
    const long stages = (long)h->B * h->N;
    k_assemble_srb<NU><<<(unsigned)((stages + 127) / 128), 128, 0, st>>>(P, q, h->srb);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h, "k_assemble_srb launch", e);
    k_factor_srb<<<(unsigned)((h->B + FAC_WARPS - 1) / FAC_WARPS), FAC_WARPS * 32, 0, st>>>(P, q.x0, h->srb, ext);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h, "k_factor_srb launch", e);

    cudaFuncAttributes fa;
    e = cudaFuncGetAttributes(&fa, k_iterate_srb<NU>);
    if (e != cudaSuccess) return fail(h, "k_iterate_srb attributes", e);
    int G = h->envs_per_cta;
    if (G > 0) {
        int threads = (G * h->N + 31) / 32 * 32;
        if (threads > 256 || iterate_smem_bytes(h->N, G, ext) > (size_t)h->smem_optin) G = 0;
    }
    if (G == 0) G = choose_G(h, fa.numRegs, ext);
    if (G == 0) {
        snprintf(h->err, sizeof h->err, "structured solver: N=%d needs %zu B of shared memory per env (limit %d)", h->N,
                 iterate_smem_bytes(h->N, 1, ext), h->smem_optin);
        return -1;
    }
    int threads = (G * h->N + 31) / 32 * 32;
    size_t smem = iterate_smem_bytes(h->N, G, ext);
    e = cudaFuncSetAttribute(k_iterate_srb<NU>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return fail(h, "k_iterate_srb smem attribute", e);
    k_iterate_srb<NU><<<(unsigned)((h->B + G - 1) / G), threads, smem, st>>>(P, h->srb, q.x0, q.mass, h->out, G, ext);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h, "k_iterate_srb launch", e);
    return 3;
}

}  // namespace

int pinmpc_launch_solve_srb(pinmpc_ctx *h, cudaStream_t st)
{
    return h->nu == 12 ? launch_t<12>(h, st) : launch_t<18>(h, st);
}
