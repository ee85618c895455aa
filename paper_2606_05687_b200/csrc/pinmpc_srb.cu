// pinmpc_srb.cu — the STRUCTURED on-chip solver (PINMPC_METHOD_SRB), the product path.
//
// One fused kernel per solve: dynamics assembly (S1), Riccati factorisation (S2) and all ADMM
// iterations (S3-S6) of one env run inside one warp with every iteration-invariant factor resident
// in shared memory.  A_k and B_k are never formed ("construction-free"):
// the single-rigid-body structure of BASELINE.json config 0 (SRB form of PAPER.md eq. (2)-(4))
//     A_k = I + dt [Theta <- R_z^T omega, p <- v, v_z <- g],     B_k = E Bh_k,
//     E = rows 6..11 (omega, v),   Bh_k = D_k Gh_k,   D_k = blkdiag(dt I_w^-1, dt/m I),
//     Gh_k u = (sum_i r_i x f_i + sum_i m_i ;  sum_i f_i)          (net wrench about the CoM)
// lets the equality-constrained step (21a) be solved EXACTLY as an LQR in the 6-D input
// w = Bh_k u (the momentum increment) instead of the nu-D input u:
//   for given w the best u is  u = u0 + Rt^-1 Bh^T S (w - Bh u0),  u0 = Rt^-1 r,  S = (Bh Rt^-1 Bh^T)^-1
//   and its cost is 1/2 (w - w0)^T S (w - w0) + const, so with P_N = Q, for k = N-1..0
//     Mh = S_k + E^T P E,  Kh = Mh^-1 E^T P A_k (6x13),  P <- [k>=1] Q + A^T P A - G^T Kh,  G = E^T P A
//   backward  g = p - s;  hh = S w0 + E^T g;  kap = Mh^-1 hh;  p <- q + A^T g - Kh^T hh
//   forward   w = -Kh x + kap;  x+ = A x + E (w + ch);  u = u0 + Rt^-1 Gh^T Lam^-1 (D^-1 w - Gh u0)
// with Lam = Gh Rt^-1 Gh^T (well conditioned; S = D^-1 Lam^-1 D^-1).  The value function P_k and
// the iterates (x,u) equal those of the dense recursion of SURVEY.md 8(c)-O2/O3 (the oracle) up to
// rounding; only 6x13 + 2 symmetric 6x6 blocks per stage are dense.
//
// Mapping (v1): CTA = one warp = one env.  Sequential passes: lane j owns row j of x / p.
// Stage-parallel phases (projection S4, dual update S5, residuals S6, u reconstruction): lane = stage.
#include "pinmpc_common.cuh"

namespace {

constexpr int NW = 2;   // 6-D wrench contacts (feet)

__host__ __device__ constexpr int sidx(int i, int j)   // packed upper triangle of a symmetric 6x6
{
    return i <= j ? (i * 6 - i * (i - 1) / 2 + (j - i)) : (j * 6 - j * (j - 1) / 2 + (i - j));
}

template <int NU>
struct Lay {
    static constexpr int NF = (NU - 12) / 3;
    static constexpr int NC = NW + NF;
    // per-stage strides in floats (odd where lanes index by stage, to stay bank-conflict free)
    static constexpr int KB = 104;        // [13][8]: Kh[0..5][j], q_j, s_j
    static constexpr int MI = 21;         // S_k during factorisation, then Mh_k^-1 (packed)
    static constexpr int LI = 21;         // Lam_k^-1 (packed)
    static constexpr int IW = 9;          // I_w packed (6), cos, sin, contact bits
    static constexpr int RR = 3 * NC + 1; // contact offsets r_i (7 / 13)
    static constexpr int RU = NU + 1;     // R ubar
    static constexpr int ZY = NU + 1;     // z, y (each)
    static constexpr int V6 = 7;          // 6-vectors: sigma0, hh/kappa, w, ch
    static constexpr int PER_STAGE = KB + MI + LI + IW + RR + RU + 2 * ZY + 4 * V6;
    static constexpr int FIXED = 3 * 172 + 80 + 80 + 40;   // P, X, Y (13x13), G, Kh (6x13), Mh (6x6)
};

// y = M x for packed symmetric 6x6
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

// In-place inverse of a packed symmetric positive definite 6x6 (Cholesky, registers only).
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
    // Li = L^-1 (lower triangular)
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
    // M^-1 = Li^T Li
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

template <int NU>
struct StageView {      // pointers into one env's shared-memory arena
    float *KB, *MI, *LI, *IW, *RR, *RU, *ZZ, *YY, *S0, *KP, *WV, *CE, *P, *X, *Y, *G, *Kh, *Mh;
    __device__ StageView(float *base, int N)
    {
        using L = Lay<NU>;
        float *p = base;
        KB = p; p += (size_t)N * L::KB;
        MI = p; p += (size_t)N * L::MI;
        LI = p; p += (size_t)N * L::LI;
        IW = p; p += (size_t)N * L::IW;
        RR = p; p += (size_t)N * L::RR;
        RU = p; p += (size_t)N * L::RU;
        ZZ = p; p += (size_t)N * L::ZY;
        YY = p; p += (size_t)N * L::ZY;
        S0 = p; p += (size_t)N * L::V6;
        KP = p; p += (size_t)N * L::V6;
        WV = p; p += (size_t)N * L::V6;
        CE = p; p += (size_t)N * L::V6;
        P = p; p += 172; X = p; p += 172; Y = p; p += 172; G = p; p += 80; Kh = p; p += 80; Mh = p;
    }
};

__device__ __forceinline__ int fcol(int i) { return i < NW ? 3 * i : 6 * NW + 3 * (i - NW); }
__device__ __forceinline__ int mcol(int i) { return 3 * NW + 3 * i; }

// u0 = Rt^-1 (R ubar + rho (z - y)) and its net wrench G0 = Gh u0 for one stage (lane-local)
template <int NU>
__device__ __forceinline__ void stage_u0(const SolveParams &P, const float *ru, const float *z, const float *y,
                                         const float *r, float *u0, float *G0)
{
    constexpr int NC = Lay<NU>::NC;
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

// D^-1 v = (I_w v_tau / dt ; m v_F / dt) with I_w packed symmetric 3x3 (xx,xy,xz,yy,yz,zz)
__device__ __forceinline__ void dinv_apply(const float *Iw, float idt, float m_dt, const float *v, float *o)
{
    o[0] = (Iw[0] * v[0] + Iw[1] * v[1] + Iw[2] * v[2]) * idt;
    o[1] = (Iw[1] * v[0] + Iw[3] * v[1] + Iw[4] * v[2]) * idt;
    o[2] = (Iw[2] * v[0] + Iw[4] * v[1] + Iw[5] * v[2]) * idt;
    o[3] = v[3] * m_dt; o[4] = v[4] * m_dt; o[5] = v[5] * m_dt;
}

template <int NU>
__global__ void __launch_bounds__(32) k_solve_srb(SolveParams P, ProblemPtrs q, OutPtrs o)
{
    using L = Lay<NU>;
    constexpr int NC = L::NC;
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ __align__(16) float smem[];
    const int lane = threadIdx.x;
    const int b = blockIdx.x;
    const int N = P.N;
    StageView<NU> V(smem, N);
    const float dt = P.dt, idt = 1.0f / P.dt;
    const float mass = q.mass[b], dtm = dt / mass, m_dt = mass / dt;
    const bool has_ext = q.ext != nullptr;

    // ------------------------------------------------------------------------------------------
    // S1  construction-free assembly: per-stage geometry, Lam^-1, S   (lane = stage)
    // ------------------------------------------------------------------------------------------
    float Ib[9], Ibi[9];
#pragma unroll
    for (int i = 0; i < 9; i++) Ib[i] = q.inertia[(long)b * 9 + i];
    inv3f(Ib, Ibi);
    for (int k = lane; k < N; k += 32) {
        const long s = (long)b * N + k;
        float sn, cs;
        sincosf(q.yaw[s], &sn, &cs);
        // I_w = R_z I_b R_z^T : same congruence as world_inertia_inv, applied to I_b
        float Iwf[9];
        world_inertia_inv(Ib, cs, sn, Iwf);
        float *iw = V.IW + k * L::IW;
        iw[0] = Iwf[0]; iw[1] = Iwf[1]; iw[2] = Iwf[2]; iw[3] = Iwf[4]; iw[4] = Iwf[5]; iw[5] = Iwf[8];
        iw[6] = cs; iw[7] = sn;
        int bits = 0;
        float r[3 * NC];
#pragma unroll
        for (int i = 0; i < NC; i++) {
            bits |= (q.contact[s * NC + i] != 0) << i;
#pragma unroll
            for (int a = 0; a < 3; a++) {
                r[3 * i + a] = q.foot_r[(s * NC + i) * 3 + a];
                V.RR[k * L::RR + 3 * i + a] = r[3 * i + a];
            }
        }
        iw[8] = __int_as_float(bits);
#pragma unroll
        for (int j = 0; j < NU; j++) {
            V.RU[k * L::RU + j] = q.u_ref ? P.Rd[j] * q.u_ref[s * NU + j] : 0.0f;
            V.ZZ[k * L::ZY + j] = 0.0f;
            V.YY[k * L::ZY + j] = 0.0f;
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
        for (int i = 0; i < 21; i++) V.LI[k * L::LI + i] = Lam[i];
        // S = D^-1 Lam^-1 D^-1,  D^-1 = blkdiag(I_w / dt, m/dt I)
        {
            const float Iw3[3][3] = { { iw[0], iw[1], iw[2] }, { iw[1], iw[3], iw[4] }, { iw[2], iw[4], iw[5] } };
            float T[3][3], S[21];
            // tau-tau block: I_w V_tt I_w / dt^2
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
            // tau-F block: I_w V_tF m / dt^2 ; F-F block: V_FF m^2 / dt^2
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
            for (int i = 0; i < 21; i++) V.MI[k * L::MI + i] = S[i];
        }
        // ch = (dt I_w^-1 tau_ext ; dt/m F_ext): the part of c_k in rows 6..11
        float ch[6] = { 0, 0, 0, 0, 0, 0 };
        if (has_ext) {
            float Wi[9];
            world_inertia_inv(Ibi, cs, sn, Wi);
            const float *e = q.ext + s * 6;
#pragma unroll
            for (int a = 0; a < 3; a++) {
                ch[a] = dt * (Wi[a * 3] * e[3] + Wi[a * 3 + 1] * e[4] + Wi[a * 3 + 2] * e[5]);
                ch[3 + a] = dtm * e[a];
            }
        }
#pragma unroll
        for (int a = 0; a < 6; a++) V.CE[k * L::V6 + a] = ch[a];
    }
    __syncwarp();

    // ------------------------------------------------------------------------------------------
    // S2  factorisation: P recursion in the 6-D input, warp-cooperative, sequential over stages
    // ------------------------------------------------------------------------------------------
    for (int i = lane; i < 169; i += 32) V.P[i] = (i / NX == i % NX) ? P.Qd[i / NX] : 0.0f;
    __syncwarp();
    for (int k = N - 1; k >= 0; k--) {
        const float cs = V.IW[k * L::IW + 6], sn = V.IW[k * L::IW + 7];
        // X = P A
        for (int e = lane; e < 169; e += 32) {
            int i = e / NX, j = e % NX;
            const float *Pi = V.P + i * NX;
            float a = Pi[j];
            if (j == 6) a += dt * (cs * Pi[0] - sn * Pi[1]);
            else if (j == 7) a += dt * (sn * Pi[0] + cs * Pi[1]);
            else if (j == 8) a += dt * Pi[2];
            else if (j >= 9 && j <= 11) a += dt * Pi[j - 6];
            else if (j == 12) a += dt * Pi[11];
            V.X[e] = a;
        }
        // Mh = S + P[6:12,6:12] ; s_k = P (E ch)
        for (int e = lane; e < 36; e += 32) {
            int i = e / 6, j = e % 6;
            V.Mh[e] = V.MI[k * L::MI + sidx(i, j)] + V.P[(6 + i) * NX + 6 + j];
        }
        float sk = 0.0f;
        if (lane < NX) {
#pragma unroll
            for (int a = 0; a < 6; a++) sk = fmaf(V.P[lane * NX + 6 + a], V.CE[k * L::V6 + a], sk);
        }
        __syncwarp();
        // Mh^-1 (lane 0, registers) ; Y = A^T X ; G = X[6:12,:]
        if (lane == 0) {
            float M[21];
#pragma unroll
            for (int i = 0; i < 6; i++)
#pragma unroll
                for (int j = i; j < 6; j++) M[sidx(i, j)] = 0.5f * (V.Mh[i * 6 + j] + V.Mh[j * 6 + i]);
            spd_inv6(M);
#pragma unroll
            for (int i = 0; i < 21; i++) V.MI[k * L::MI + i] = M[i];
        }
        for (int e = lane; e < 169; e += 32) {
            int i = e / NX, j = e % NX;
            float a = V.X[e];
            if (i == 6) a += dt * (cs * V.X[0 * NX + j] - sn * V.X[1 * NX + j]);
            else if (i == 7) a += dt * (sn * V.X[0 * NX + j] + cs * V.X[1 * NX + j]);
            else if (i == 8) a += dt * V.X[2 * NX + j];
            else if (i >= 9 && i <= 11) a += dt * V.X[(i - 6) * NX + j];
            else if (i == 12) a += dt * V.X[11 * NX + j];
            V.Y[e] = a;
        }
        __syncwarp();
        // Kh = Mh^-1 G
        for (int e = lane; e < 78; e += 32) {
            int i = e / NX, j = e % NX;
            float a = 0.0f;
#pragma unroll
            for (int l = 0; l < 6; l++) a = fmaf(V.MI[k * L::MI + sidx(i, l)], V.X[(6 + l) * NX + j], a);
            V.Kh[e] = a;
        }
        __syncwarp();
        // store the sequential block: Kh^T, q_k, s_k
        if (lane < NX) {
            float *kb = V.KB + k * L::KB + lane * 8;
#pragma unroll
            for (int i = 0; i < 6; i++) kb[i] = V.Kh[i * NX + lane];
            kb[6] = (k >= 1) ? P.Qd[lane] * q.x_ref[((long)b * N + k - 1) * NX + lane] : 0.0f;
            kb[7] = sk;
        }
        // Z = Y - G^T Kh  (into X's storage is unsafe: G lives there) -> into P after symmetrisation
        float zloc[6];
        int cnt = 0;
        for (int e = lane; e < 169; e += 32, cnt++) {
            int i = e / NX, j = e % NX;
            float a = V.Y[e];
#pragma unroll
            for (int l = 0; l < 6; l++) a = fmaf(-V.X[(6 + l) * NX + i], V.Kh[l * NX + j], a);
            zloc[cnt] = a;
        }
        __syncwarp();
        cnt = 0;
        for (int e = lane; e < 169; e += 32, cnt++) V.Y[e] = zloc[cnt];
        __syncwarp();
        for (int e = lane; e < 169; e += 32) {
            int i = e / NX, j = e % NX;
            V.P[e] = 0.5f * (V.Y[i * NX + j] + V.Y[j * NX + i]) + ((k >= 1 && i == j) ? P.Qd[i] : 0.0f);
        }
        __syncwarp();
    }

    // ------------------------------------------------------------------------------------------
    // S3-S6  ADMM iterations
    // ------------------------------------------------------------------------------------------
    // per-lane constants of the structured A: (A^T g)_j = g_j + ca g[sa] + cb g[sb], same for A x
    int bsa = 0, bsb = 0, fsa = 0, fsb = 0;
    float b_c1 = 0, b_cc = 0, b_cs = 0, b_dc = 0, b_ds = 0;      // backward: ca = b_c1 + b_cc cs + b_cs sn ; cb = b_dc cs + b_ds sn
    float f_c1 = 0, f_cc = 0, f_cs = 0, f_dc = 0, f_ds = 0;
    if (lane == 6) { bsa = 0; bsb = 1; b_cc = dt; b_ds = -dt; }
    else if (lane == 7) { bsa = 0; bsb = 1; b_cs = dt; b_dc = dt; }
    else if (lane >= 8 && lane <= 11) { bsa = lane - 6; b_c1 = dt; }
    else if (lane == 12) { bsa = 11; b_c1 = dt; }
    if (lane == 0) { fsa = 6; fsb = 7; f_cc = dt; f_ds = dt; }
    else if (lane == 1) { fsa = 6; fsb = 7; f_cs = -dt; f_dc = dt; }
    else if (lane >= 2 && lane <= 5) { fsa = lane + 6; f_c1 = dt; }
    else if (lane == 11) { fsa = 12; f_c1 = dt; }
    const int wsrc = (lane >= 6 && lane < 12) ? lane - 6 : 0;
    const float Qd_l = lane < NX ? P.Qd[lane] : 0.0f;
    const float x0_l = lane < NX ? q.x0[(long)b * NX + lane] : 0.0f;
    const float pN_l = lane < NX ? Qd_l * q.x_ref[((long)b * N + N - 1) * NX + lane] : 0.0f;
    const bool tol_mode = (P.eps_abs > 0.0f || P.eps_rel > 0.0f) && P.check_every > 0;

    // sigma0 for the first iteration (z = y = 0)
    auto stage_sigma0 = [&](int k) {
        float u0[NU], G0[6], l0[6], s0[6];
        stage_u0<NU>(P, V.RU + k * L::RU, V.ZZ + k * L::ZY, V.YY + k * L::ZY, V.RR + k * L::RR, u0, G0);
        symv6(V.LI + k * L::LI, G0, l0);
        dinv_apply(V.IW + k * L::IW, idt, m_dt, l0, s0);
#pragma unroll
        for (int a = 0; a < 6; a++) V.S0[k * L::V6 + a] = s0[a];
    };
    for (int k = lane; k < N; k += 32) stage_sigma0(k);
    __syncwarp();

    float rp = 0.0f, rd = 0.0f;
    int done = 0;
    for (int it = 0; it < P.iters; it++) {
        const bool is_check = tol_mode && ((it + 1) % P.check_every == 0);
        const bool emit = (it == P.iters - 1) || is_check;
        // ---- backward vector pass (sequential over stages; lane j = row j) ----------------------
        float p = pN_l;
        for (int k = N - 1; k >= 0; k--) {
            const float4 *kb4 = reinterpret_cast<const float4 *>(V.KB + k * L::KB + (lane < NX ? lane : 0) * 8);
            float4 k0 = kb4[0], k1 = kb4[1];            // Kh[0..3][j] | Kh[4][j], Kh[5][j], q_j, s_j
            const float cs = V.IW[k * L::IW + 6], sn = V.IW[k * L::IW + 7];
            float g = p - k1.w;
            float hh = g + ((lane >= 6 && lane < 12) ? V.S0[k * L::V6 + lane - 6] : 0.0f);   // lanes 6..11
            if (lane >= 6 && lane < 12) V.KP[k * L::V6 + lane - 6] = hh;
            float h0 = __shfl_sync(FULL, hh, 6), h1 = __shfl_sync(FULL, hh, 7), h2 = __shfl_sync(FULL, hh, 8);
            float h3 = __shfl_sync(FULL, hh, 9), h4 = __shfl_sync(FULL, hh, 10), h5 = __shfl_sync(FULL, hh, 11);
            float ga = __shfl_sync(FULL, g, bsa), gb = __shfl_sync(FULL, g, bsb);
            float ca = fmaf(b_cc, cs, fmaf(b_cs, sn, b_c1)), cb = fmaf(b_dc, cs, b_ds * sn);
            float acc = k1.z + g;
            acc = fmaf(ca, ga, acc); acc = fmaf(cb, gb, acc);
            float t0 = fmaf(k0.x, h0, fmaf(k0.y, h1, k0.z * h2));
            float t1 = fmaf(k0.w, h3, fmaf(k1.x, h4, k1.y * h5));
            p = acc - (t0 + t1);
        }
        __syncwarp();
        // ---- kappa = Mh^-1 hh (lane = stage) ------------------------------------------------------
        for (int k = lane; k < N; k += 32) {
            float h[6], kp[6];
#pragma unroll
            for (int a = 0; a < 6; a++) h[a] = V.KP[k * L::V6 + a];
            symv6(V.MI + k * L::MI, h, kp);
#pragma unroll
            for (int a = 0; a < 6; a++) V.KP[k * L::V6 + a] = kp[a];
        }
        __syncwarp();
        // ---- forward rollout (sequential; lane j = row j of x, lanes 0..5 also own w_i) -----------
        float x = x0_l;
        for (int k = 0; k < N; k++) {
            const float *kb = V.KB + k * L::KB;
            const float cs = V.IW[k * L::IW + 6], sn = V.IW[k * L::IW + 7];
            float w = (lane < 6) ? V.KP[k * L::V6 + lane] : 0.0f;
            const int li = lane < 6 ? lane : 0;
#pragma unroll
            for (int j = 0; j < NX; j++) {
                float xj = __shfl_sync(FULL, x, j);
                w = fmaf(-kb[j * 8 + li], xj, w);
            }
            if (lane < 6) V.WV[k * L::V6 + lane] = w;
            float wc = w + ((lane < 6) ? V.CE[k * L::V6 + lane] : 0.0f);
            float wj = __shfl_sync(FULL, wc, wsrc);
            float xa = __shfl_sync(FULL, x, fsa), xb = __shfl_sync(FULL, x, fsb);
            float ca = fmaf(f_cc, cs, fmaf(f_cs, sn, f_c1)), cb = fmaf(f_dc, cs, f_ds * sn);
            float xn = fmaf(ca, xa, fmaf(cb, xb, x));
            if (lane >= 6 && lane < 12) xn += wj;
            x = xn;
            if (emit && lane < NX) o.x[((long)b * N + k) * NX + lane] = x;
        }
        __syncwarp();
        // ---- u reconstruction, projection, dual update, residuals (lane = stage) -------------------
        float rp_l = 0.0f, rd_l = 0.0f, un_l = 0.0f, zn_l = 0.0f, yn_l = 0.0f;
        for (int k = lane; k < N; k += 32) {
            float u0[NU], G0[6], wv[6], dl[6], lam[6], z[NU], y[NU], r[3 * NC];
#pragma unroll
            for (int j = 0; j < NU; j++) { z[j] = V.ZZ[k * L::ZY + j]; y[j] = V.YY[k * L::ZY + j]; }
#pragma unroll
            for (int j = 0; j < 3 * NC; j++) r[j] = V.RR[k * L::RR + j];
            stage_u0<NU>(P, V.RU + k * L::RU, z, y, r, u0, G0);
#pragma unroll
            for (int a = 0; a < 6; a++) wv[a] = V.WV[k * L::V6 + a];
            dinv_apply(V.IW + k * L::IW, idt, m_dt, wv, dl);
#pragma unroll
            for (int a = 0; a < 6; a++) dl[a] -= G0[a];
            symv6(V.LI + k * L::LI, dl, lam);
            // u = u0 + Rt^-1 Gh^T lam :  f_i += lam_tau x r_i + lam_F ;  m_i += lam_tau
            float u[NU];
#pragma unroll
            for (int i = 0; i < NC; i++) {
                float rx = r[3 * i], ry = r[3 * i + 1], rz = r[3 * i + 2];
                float c0 = lam[1] * rz - lam[2] * ry + lam[3];
                float c1 = lam[2] * rx - lam[0] * rz + lam[4];
                float c2 = lam[0] * ry - lam[1] * rx + lam[5];
                int fc = fcol(i);
                u[fc] = u0[fc] + c0 / (P.Rd[fc] + P.rho);
                u[fc + 1] = u0[fc + 1] + c1 / (P.Rd[fc + 1] + P.rho);
                u[fc + 2] = u0[fc + 2] + c2 / (P.Rd[fc + 2] + P.rho);
                if (i < NW) {
                    int mc = mcol(i);
#pragma unroll
                    for (int a = 0; a < 3; a++) u[mc + a] = u0[mc + a] + lam[a] / (P.Rd[mc + a] + P.rho);
                }
            }
            // projection (S4), dual update (S5), residuals (S6)
            const int bits = __float_as_int(V.IW[k * L::IW + 8]);
            float zn[NU];
#pragma unroll
            for (int i = 0; i < NC; i++) {
                const bool on = (bits >> i) & 1;
                int fc = fcol(i);
                if (i < NW) {
                    int mc = mcol(i);
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
#pragma unroll
            for (int j = 0; j < NU; j++) {
                float yn = y[j] + u[j] - zn[j];
                rp_l = fmaxf(rp_l, fabsf(u[j] - zn[j]));
                rd_l = fmaxf(rd_l, fabsf(zn[j] - z[j]));
                un_l = fmaxf(un_l, fabsf(u[j])); zn_l = fmaxf(zn_l, fabsf(zn[j])); yn_l = fmaxf(yn_l, fabsf(yn));
                V.ZZ[k * L::ZY + j] = zn[j];
                V.YY[k * L::ZY + j] = yn;
                if (emit) o.u[((long)b * N + k) * NU + j] = u[j];
            }
            stage_sigma0(k);           // sigma0 of the next iteration from the new z, y
        }
        __syncwarp();
        rp = warp_max(rp_l); rd = P.rho * warp_max(rd_l);
        done = it + 1;
        if (is_check) {
            float sc = fmaxf(warp_max(un_l), warp_max(zn_l)), ys = warp_max(yn_l);
            if (rp <= P.eps_abs + P.eps_rel * sc && rd <= P.eps_abs + P.eps_rel * P.rho * ys) break;
        }
    }
    for (int k = lane; k < N; k += 32)
#pragma unroll
        for (int j = 0; j < NU; j++) {
            o.z[((long)b * N + k) * NU + j] = V.ZZ[k * L::ZY + j];
            o.y[((long)b * N + k) * NU + j] = V.YY[k * L::ZY + j];
        }
    if (lane == 0) { o.r_prim[b] = rp; o.r_dual[b] = rd; o.iters_done[b] = done; }
}

template <int NU>
size_t smem_bytes_t(int N) { return ((size_t)Lay<NU>::PER_STAGE * N + Lay<NU>::FIXED) * sizeof(float); }

template <int NU>
int launch_t(pinmpc_ctx *h, cudaStream_t st)
{
    size_t smem = smem_bytes_t<NU>(h->N);
    if (smem > (size_t)h->smem_optin) {
        snprintf(h->err, sizeof h->err, "structured solver: N=%d needs %zu B of shared memory per env (limit %d)", h->N,
                 smem, h->smem_optin);
        return -1;
    }
    cudaError_t e = cudaFuncSetAttribute(k_solve_srb<NU>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) {
        k_solve_srb<NU><<<h->B, 32, smem, st>>>(make_params(h), make_problem_ptrs(h), h->out);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        h->sticky = e;
        snprintf(h->err, sizeof h->err, "k_solve_srb launch: %s", cudaGetErrorString(e));
        return -1;
    }
    return 1;
}

}  // namespace

size_t pinmpc_srb_smem_bytes(int nu, int N) { return nu == 12 ? smem_bytes_t<12>(N) : smem_bytes_t<18>(N); }

int pinmpc_launch_solve_srb(pinmpc_ctx *h, cudaStream_t st)
{
    return h->nu == 12 ? launch_t<12>(h, st) : launch_t<18>(h, st);
}
