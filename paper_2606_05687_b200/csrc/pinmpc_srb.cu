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
//   k_iterate_srb   S3-6 the SEQUENTIAL-PASS iteration kernel (pinmpc_set_horizon_chunks(h, 1), and the fallback for
//                        shapes the chunked kernel of pinmpc_tmem.cu cannot hold): one CTA per G envs, all ADMM
//                        iterations with Kh and the exchange vectors in shared memory; PW pass warps run the two
//                        N-step recursions (six lanes per env, five envs per warp), the stage threads own two
//                        stages each with z, y in registers and stream the stage records from L2.
#include <mutex>

#include "pinmpc_srb_math.cuh"

namespace {

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
    float rb[pinmpc_rb_width(NU)];
#pragma unroll
    for (int i = 0; i < pinmpc_rb_width(NU); i++) rb[i] = 0.0f;
#pragma unroll
    for (int i = 0; i < 6; i++) rb[6 + i] = iw[i];

    int bits = 0;
    float r[3 * NC];
#pragma unroll
    for (int i = 0; i < NC; i++) {
        bits |= (q.contact[s * NC + i] != 0) << i;
#pragma unroll
        for (int a = 0; a < 3; a++) {
            r[3 * i + a] = q.foot_r[(s * NC + i) * 3 + a];
            rb[12 + 3 * i + a] = r[3 * i + a];
        }
    }
    rb[12 + 3 * NC + NU] = __int_as_float(bits);
#pragma unroll
    for (int j = 0; j < NU; j++) rb[12 + 3 * NC + j] = q.u_ref ? P.tR[j] * P.Rd[j] * q.u_ref[s * NU + j] : 0.0f;
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
    // T^-1, T = Lam_tt - Lam_tF Lam_FF^-1 Lam_Ft (Schur complement; Lam_FF = diag(1 / phi_inv) for every stage):
    // the iteration kernel applies Lam^-1 through T^-1 and r (6 + 0 words per stage instead of 21)
    {
        float T[6], TI[6];
#pragma unroll
        for (int x = 0; x < 3; x++)
#pragma unroll
            for (int y = x; y < 3; y++) {
                float a = Lam[sidx(x, y)];
#pragma unroll
                for (int l = 0; l < 3; l++) a = fmaf(-Lam[sidx(x, 3 + l)] * P.phi_inv[l], Lam[sidx(y, 3 + l)], a);
                T[x * 3 - x * (x - 1) / 2 + (y - x)] = a;
            }
        // symmetric 3x3 inverse (xx,xy,xz,yy,yz,zz)
        const float c00 = T[3] * T[5] - T[4] * T[4], c01 = T[2] * T[4] - T[1] * T[5], c02 = T[1] * T[4] - T[2] * T[3];
        const float id = 1.0f / (T[0] * c00 + T[1] * c01 + T[2] * c02);
        TI[0] = c00 * id; TI[1] = c01 * id; TI[2] = c02 * id;
        TI[3] = (T[0] * T[5] - T[2] * T[2]) * id; TI[4] = (T[1] * T[2] - T[0] * T[4]) * id;
        TI[5] = (T[0] * T[3] - T[1] * T[1]) * id;
#pragma unroll
        for (int i = 0; i < 6; i++) rb[i] = TI[i];
    }
    spd_inv6(Lam);                                   // Lam^-1 (for S below)
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
        // S_k as six float4 groups, group-major (the layout of the stage records): coalesced here, six 16-byte loads per
        // stage in the factorisation
        {
            float4 *MI4 = reinterpret_cast<float4 *>(W.MI);
#pragma unroll
            for (int g = 0; g < 6; g++)
                MI4[(long)g * st + s] = make_float4(S[4 * g], 4 * g + 1 < 21 ? S[4 * g + 1] : 0.0f, 4 * g + 2 < 21 ? S[4 * g + 2] : 0.0f,
                                                    4 * g + 3 < 21 ? S[4 * g + 3] : 0.0f);
        }
    }
    // the stage record of the iteration kernel: float4 component-major
    {
        float4 *RB4 = reinterpret_cast<float4 *>(W.RB);
#pragma unroll
        for (int c = 0; c < pinmpc_rb_width(NU) / 4; c++)
            RB4[(long)c * st + s] = make_float4(rb[4 * c], rb[4 * c + 1], rb[4 * c + 2], rb[4 * c + 3]);
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
// S2  factorisation: TWO envs per warp (lanes 0-15 and 16-31), sequential over stages.  Lane hl < 13 of a half owns
// row hl of the 13x13 matrices P and X = P A of its env (rows 20 floats apart in shared memory, float4 accesses, no
// index arithmetic in the loop).  The symmetric 6x6 Mh is inverted by sweeps on the packed 21 elements, one element
// per lane 0..20 of the whole warp, for one env after the other (the only part that is not packed).  With one env per
// warp 13 of 32 lanes worked: the kernel is bound by issue slots and shared-memory wavefronts, so packing halves it.
// ---------------------------------------------------------------------------------------------
constexpr int FAC_WARPS = 4;                        // warps per CTA (8 envs)
constexpr int FAC_EPW = 2;                          // envs per warp
constexpr int FAC_LD = 20;                          // padded row length: rows 80 B apart, the float4 row accesses of eight lanes hit distinct banks
constexpr int FAC_SMEM = 13 * FAC_LD + 13 * FAC_LD + 6 * FAC_LD + 24;   // floats per env: P, X, Kh, Mh^-1

__global__ void __launch_bounds__(FAC_WARPS * 32, 4) k_factor_srb(SolveParams P, const float *__restrict__ x0, SrbWs W, int has_ext, int C, float *__restrict__ Psi)
{
    __shared__ __align__(16) float sm_all[FAC_WARPS * FAC_EPW * FAC_SMEM];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int hf = lane >> 4, hl = lane & 15, hb = 16 * hf;          // half of the warp, lane inside it, its first lane
    const int bw = (blockIdx.x * FAC_WARPS + wib) * FAC_EPW;         // first env of the warp
    if (bw >= P.B) return;
    const bool pair = bw + 1 < P.B;                                  // a last odd env: half 1 shadows it (no stores)
    const int b = bw + (pair ? hf : 0);
    const bool live = hf == 0 || pair;
    // (plain arithmetic on the __shared__ array, so that the accesses compile to LDS / STS: a pointer picked from an array
    // of pointers made them generic loads, which go through the global-memory queue)
    float *sP = sm_all + (wib * FAC_EPW + hf) * FAC_SMEM, *sX = sP + 13 * FAC_LD, *sK = sX + 13 * FAC_LD, *sM = sK + 6 * FAC_LD;
    const int N = P.N;
    const long st = (long)P.B * N;
    const float dt = P.dt;
    const float x12 = x0[(long)b * NX + 12];
    const int row = hl < NX ? hl : 0;                 // lanes >= 13 of a half shadow row 0 (no stores)
    const bool rown = hl < NX;

    // A^T X: row i of A^T X = X[i] + ea X[ra] + eb X[rb]  (rows 6..12 pick up dt * rows of X)
    const int ra = row == 6 || row == 7 ? 0 : (row == 8 ? 2 : (row >= 9 && row <= 11 ? row - 6 : (row == 12 ? 11 : 0)));
    const int rb = row == 6 || row == 7 ? 1 : ra;
    const float qd = rown ? P.Qd[row] : 0.0f;

    // P_N = Q
    if (rown) {
#pragma unroll
        for (int c = 0; c < 4; c++) {
            float4 v = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            if (row == 4 * c) v.x = qd; else if (row == 4 * c + 1) v.y = qd; else if (row == 4 * c + 2) v.z = qd; else if (row == 4 * c + 3) v.w = qd;
            *reinterpret_cast<float4 *>(sP + row * FAC_LD + 4 * c) = v;
        }
    }
    __syncwarp();
    const int jl = hl < 12 ? hl : 0;
    float pc = W.qv[((long)b * (N + 1) + N) * 12 + jl];     // pc_N = q_N
    const long sq[FAC_EPW] = { (long)bw * N, (long)(bw + (pair ? 1 : 0)) * N };     // stage 0 of the warp's two envs

    // prefetch stage N-1
    long s = (long)b * N + N - 1;
    float cs_n = W.cs[s * 2], sn_n = W.cs[s * 2 + 1];
    const float4 *MI4 = reinterpret_cast<const float4 *>(W.MI);
    float4 S_n[6];                                    // S_k of the own env, all 21 packed elements in every lane (broadcast loads)
#pragma unroll
    for (int g = 0; g < 6; g++) S_n[g] = MI4[(long)g * st + s];
    float ch_n = (has_ext && hl < 6) ? W.c6[s * 6 + hl] : 0.0f;
    float q_n = N >= 2 ? W.qv[((long)b * (N + 1) + N - 1) * 12 + jl] : 0.0f;      // q_k of the stage being processed
    // chunk operators of the chunked iteration kernel, formed on the way (C > 2): lane hl < 12 carries row hl of
    // Psi_c = Phi_{k0+len-1} ... Phi_{k0} of the chunk the walk is in, row <- row Phi_k, and stores it at the chunk's first
    // stage.  Psi [B][C-2][12][12] for the inner chunks c = 1 .. C-2.  (This chain is independent of the Riccati chain and
    // fills issue slots the latter leaves empty; as a kernel of its own it took 43 us.)
    int pc_c = C - 1, pc_k0 = 0, pc_len = 0;
    if (C > 2) tm_chunk(N, C, pc_c, pc_k0, pc_len);
    float pa[6], pb[6];
#pragma unroll
    for (int j = 0; j < 6; j++) { pa[j] = 0.0f; pb[j] = 0.0f; }
    for (int k = N - 1; k >= 0; k--) {
        s = (long)b * N + k;
        const float cs = cs_n, sn = sn_n, chl = ch_n, qk12 = k >= 1 ? q_n : 0.0f;
        // ---- Mh = S + P[6:12,6:12], packed upper triangle, in every lane of the half (rows 6..11 of P, columns 4..11: two
        // aligned float4 per row, the block starts at column 6)
        float M[21];
#pragma unroll
        for (int i = 0; i < 6; i++) {
            const float4 lo = *reinterpret_cast<const float4 *>(sP + (6 + i) * FAC_LD + 4), hi = *reinterpret_cast<const float4 *>(sP + (6 + i) * FAC_LD + 8);
            const float pr[6] = { lo.z, lo.w, hi.x, hi.y, hi.z, hi.w };
#pragma unroll
            for (int j = i; j < 6; j++) {
                const float4 sg = S_n[sidx(i, j) >> 2];
                const int w = sidx(i, j) & 3;
                M[sidx(i, j)] = (w == 0 ? sg.x : (w == 1 ? sg.y : (w == 2 ? sg.z : sg.w))) + pr[j];
            }
        }
        if (k > 1) q_n = W.qv[((long)b * (N + 1) + k - 1) * 12 + jl];
        if (k > 0) {
            cs_n = W.cs[(s - 1) * 2]; sn_n = W.cs[(s - 1) * 2 + 1];
#pragma unroll
            for (int g = 0; g < 6; g++) S_n[g] = MI4[(long)g * st + s - 1];
            ch_n = (has_ext && hl < 6) ? W.c6[(s - 1) * 6 + hl] : 0.0f;
        }
        // ---- X = P A, row `row`:  columns 6..12 pick up dt * (R_z^T | I | e_11) combinations of columns 0..5, 11
        float xr[16];
        {
            const float4 *Pr = reinterpret_cast<const float4 *>(sP + row * FAC_LD);
            const float4 p0 = Pr[0], p1 = Pr[1], p2 = Pr[2], p3 = Pr[3];
            xr[0] = p0.x; xr[1] = p0.y; xr[2] = p0.z; xr[3] = p0.w; xr[4] = p1.x; xr[5] = p1.y;
            xr[6] = fmaf(dt, cs * p0.x - sn * p0.y, p1.z);
            xr[7] = fmaf(dt, sn * p0.x + cs * p0.y, p1.w);
            xr[8] = fmaf(dt, p0.z, p2.x);
            xr[9] = fmaf(dt, p0.w, p2.y); xr[10] = fmaf(dt, p1.x, p2.z); xr[11] = fmaf(dt, p1.y, p2.w);
            xr[12] = fmaf(dt, p2.w, p3.x);
            xr[13] = xr[14] = xr[15] = 0.0f;
            if (rown) {
                float4 *Xr = reinterpret_cast<float4 *>(sX + row * FAC_LD);
                Xr[0] = make_float4(xr[0], xr[1], xr[2], xr[3]); Xr[1] = make_float4(xr[4], xr[5], xr[6], xr[7]);
                Xr[2] = make_float4(xr[8], xr[9], xr[10], xr[11]); Xr[3] = make_float4(xr[12], 0.0f, 0.0f, 0.0f);
            }
        }
        // ---- s_k = P (E ch)
        float sk = 0.0f;
        if (has_ext) {
#pragma unroll
            for (int a = 0; a < 6; a++) sk = fmaf(sP[row * FAC_LD + 6 + a], __shfl_sync(FULL, chl, hb + a), sk);
        }
        // ---- Mh^-1 by symmetric sweeps (-Mh^-1 after six pivots), redundantly in the registers of every lane: no exchange
        // between lanes inside this chain, the longest of a stage (with one element per lane and three shuffles per pivot
        // it was 40 % of the kernel's time).  The reciprocal without the slow path of an IEEE division: d > 0 is a pivot
        // of an SPD matrix, 1 ulp is far inside the parity budget.
#pragma unroll
        for (int p = 0; p < 6; p++) {
            const float id = __fdividef(1.0f, M[sidx(p, p)]);
            float t[6], Mn[21];
#pragma unroll
            for (int i = 0; i < 6; i++) t[i] = M[sidx(i, p)] * id;
#pragma unroll
            for (int i = 0; i < 6; i++)
#pragma unroll
                for (int j = i; j < 6; j++)
                    Mn[sidx(i, j)] = (i == p && j == p) ? -id : (i == p ? t[j] : (j == p ? t[i] : fmaf(-t[i], M[sidx(p, j)], M[sidx(i, j)])));
#pragma unroll
            for (int i = 0; i < 21; i++) M[i] = Mn[i];
        }
#pragma unroll
        for (int i = 0; i < 21; i++) M[i] = -M[i];
        if (hl == 0) {                                       // one lane per env publishes Mh^-1 (for the record and the vector pass)
#pragma unroll
            for (int c = 0; c < 5; c++) *reinterpret_cast<float4 *>(sM + 4 * c) = make_float4(M[4 * c], M[4 * c + 1], M[4 * c + 2], M[4 * c + 3]);
            sM[20] = M[20];
        }
        __syncwarp();
        // ---- Kh = Mh^-1 X[6:12,:], column `row`;  xc = X[6..11][row] = G[:, row] is reused for the P update
        float xc[6], kc[6];
#pragma unroll
        for (int l = 0; l < 6; l++) xc[l] = sX[(6 + l) * FAC_LD + row];
        symv6(M, xc, kc);
        if (lane < 21) {                                     // the packed Mh^-1 of both envs -> stage records
#pragma unroll
            for (int q = 0; q < FAC_EPW; q++)
                if (q == 0 || pair) W.RA[pinmpc_rec_index(lane, st, sq[q] + k)] = sm_all[(wib * FAC_EPW + q) * FAC_SMEM + 32 * FAC_LD + lane];
        }
        if (rown) {
#pragma unroll
            for (int r = 0; r < 6; r++) sK[r * FAC_LD + row] = kc[r];
            if (row < 12 && live) {
                const int pos = row < 6 ? 2 * row : 2 * (row - 6) + 1;
#pragma unroll
                for (int r = 0; r < 6; r++) W.Kh[s * 72 + r * 12 + pos] = kc[r];
            }
        }
        __syncwarp();
        if (C > 2) {                                         // (uniform)
            if (k < pc_k0) { pc_c--; tm_chunk(N, C, pc_c, pc_k0, pc_len); }
            if (pc_c >= 1 && pc_c <= C - 2) {
                if (k == pc_k0 + pc_len - 1) {
#pragma unroll
                    for (int j = 0; j < 6; j++) { pa[j] = (hl == j) ? 1.0f : 0.0f; pb[j] = (hl == 6 + j) ? 1.0f : 0.0f; }
                }
                //   (row Phi)_a = row_a + row_b Kn_a ;  (row Phi)_b = dt row_a Rot + row_b + row_b Kn_b,  Kn = -Kh
                float na[6], nb[6];
                nb[0] = fmaf(dt, cs * pa[0] - sn * pa[1], pb[0]);
                nb[1] = fmaf(dt, sn * pa[0] + cs * pa[1], pb[1]);
#pragma unroll
                for (int j = 2; j < 6; j++) nb[j] = fmaf(dt, pa[j], pb[j]);
#pragma unroll
                for (int j = 0; j < 6; j++) na[j] = pa[j];
#pragma unroll
                for (int r = 0; r < 6; r++) {
                    const float4 k0v = *reinterpret_cast<const float4 *>(sK + r * FAC_LD), k1v = *reinterpret_cast<const float4 *>(sK + r * FAC_LD + 4),
                                 k2v = *reinterpret_cast<const float4 *>(sK + r * FAC_LD + 8);
                    const float m = -pb[r];
                    na[0] = fmaf(m, k0v.x, na[0]); na[1] = fmaf(m, k0v.y, na[1]); na[2] = fmaf(m, k0v.z, na[2]); na[3] = fmaf(m, k0v.w, na[3]);
                    na[4] = fmaf(m, k1v.x, na[4]); na[5] = fmaf(m, k1v.y, na[5]); nb[0] = fmaf(m, k1v.z, nb[0]); nb[1] = fmaf(m, k1v.w, nb[1]);
                    nb[2] = fmaf(m, k2v.x, nb[2]); nb[3] = fmaf(m, k2v.y, nb[3]); nb[4] = fmaf(m, k2v.z, nb[4]); nb[5] = fmaf(m, k2v.w, nb[5]);
                }
#pragma unroll
                for (int j = 0; j < 6; j++) { pa[j] = na[j]; pb[j] = nb[j]; }
                if (k == pc_k0 && hl < 12 && live) {
                    float4 *o = reinterpret_cast<float4 *>(Psi + (((long)b * (C - 2) + pc_c - 1) * 12 + hl) * 12);
                    o[0] = make_float4(pa[0], pa[1], pa[2], pa[3]); o[1] = make_float4(pa[4], pa[5], pb[0], pb[1]); o[2] = make_float4(pb[2], pb[3], pb[4], pb[5]);
                }
            }
        }
        // ---- iteration-invariant part of the backward vector pass (response to q and s, sigma0 = 0):
        //   g = pc - s_k ; hq_k = E^T g ; pc <- q_k + A^T g - Kh^T hq_k        (lane hl < 12 of the half holds pc_j)
        // The iteration kernel runs the sigma0-driven part only; hq_k enters kappa_k through kg_k.
        {
            const float g = pc - sk;
            const float g_lo = __shfl_sync(FULL, g, hb + (hl >= 6 ? hl - 6 : hl));
            const float g_nb = __shfl_sync(FULL, g, hb + (hl >= 6 ? (hl - 6) ^ 1 : hl));
            float acc = 0.0f, mh = 0.0f;
            const int il = hl < 6 ? hl : 0;
#pragma unroll
            for (int r = 0; r < 6; r++) {
                const float hr = __shfl_sync(FULL, g, hb + 6 + r);
                acc = fmaf(kc[r], hr, acc);                 // kc = Kh[:, hl] for hl < 13
                mh = fmaf(sM[sidx(il, r)], hr, mh);
            }
            // constant part of kappa_k = Mh^-1 hh_k - Kh[:,12] x_12 :  kg_k = Kh[:,12] x_12 - Mh^-1 hq_k
            if (hl < 6 && live) W.RA[pinmpc_rec_index(21 + hl, st, s)] = fmaf(sK[hl * FAC_LD + 12], x12, -mh);
            float atg = g;
            if (hl == 6) atg = fmaf(dt, cs * g_lo - sn * g_nb, g);
            else if (hl == 7) atg = fmaf(dt, cs * g_lo + sn * g_nb, g);
            else if (hl >= 8 && hl < 12) atg = fmaf(dt, g_lo, g);
            pc = qk12 + atg - acc;
        }
        // ---- P <- [k>=1] Q + A^T X - G^T Kh, row `row`, four columns at a time
        {
            const float ea = row == 6 ? dt * cs : (row == 7 ? dt * sn : (row >= 8 ? dt : 0.0f));
            const float eb = row == 6 ? -dt * sn : (row == 7 ? dt * cs : 0.0f);
            const float qk = k >= 1 ? qd : 0.0f;
#pragma unroll
            for (int c = 0; c < 4; c++) {
                const float4 xa = *reinterpret_cast<const float4 *>(sX + ra * FAC_LD + 4 * c);
                const float4 xb = *reinterpret_cast<const float4 *>(sX + rb * FAC_LD + 4 * c);
                float4 o;
                o.x = fmaf(ea, xa.x, fmaf(eb, xb.x, xr[4 * c])); o.y = fmaf(ea, xa.y, fmaf(eb, xb.y, xr[4 * c + 1]));
                o.z = fmaf(ea, xa.z, fmaf(eb, xb.z, xr[4 * c + 2])); o.w = fmaf(ea, xa.w, fmaf(eb, xb.w, xr[4 * c + 3]));
#pragma unroll
                for (int l = 0; l < 6; l++) {
                    const float4 kv = *reinterpret_cast<const float4 *>(sK + l * FAC_LD + 4 * c);
                    o.x = fmaf(-xc[l], kv.x, o.x); o.y = fmaf(-xc[l], kv.y, o.y);
                    o.z = fmaf(-xc[l], kv.z, o.z); o.w = fmaf(-xc[l], kv.w, o.w);
                }
                o.x += row == 4 * c ? qk : 0.0f; o.y += row == 4 * c + 1 ? qk : 0.0f;
                o.z += row == 4 * c + 2 ? qk : 0.0f; o.w += row == 4 * c + 3 ? qk : 0.0f;
                // upper triangle (j >= row), mirrored: P stays exactly symmetric over long horizons
                const float ov[4] = { o.x, o.y, o.z, o.w };
#pragma unroll
                for (int d = 0; d < 4; d++) {
                    const int j = 4 * c + d;
                    if (j < NX && rown && j >= row) { sP[row * FAC_LD + j] = ov[d]; sP[j * FAC_LD + row] = ov[d]; }
                }
            }
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------
// S3-S6  ADMM iterations: one CTA per G envs, every factor on chip (v3)
// ---------------------------------------------------------------------------------------------
// STAGE threads own one (env, stage) each and keep the stage-local data (T^-1, I_w, r, ubar, z, y)
// in registers for all iterations ("stage work": u from w, projection S4, dual update S5,
// residuals S6, sigma0 of the next iteration, kappa).  The first PW warps of the CTA are PASS warps:
// they run the two sequential vector recursions of up to five envs each, six lanes per env
// (lane = 6 e + i), exchanging the 6-D quantities with warp shuffles; the gains stream from the
// env's shared-memory arena through explicit ld.shared with immediate offsets, one stage ahead.
//
// Shared-memory arena of one env (offsets in floats):
//   Kn [N][6][6][2]  pairs -(Kh[r][j], Kh[r][6+j]): row r contiguous (forward pass, lane = row,
//                    3 x LDS.128), pair [r][i] (backward pass, lane = column pair, 6 x LDS.64)
//   X  [N][8]        exchange record [v0 v1 cos sin v2 v3 v4 v5], v: sigma0 -> hh -> kappa -> w;
//                    cos, sin of the linearisation yaw ride along (one LDS.128 serves lanes 0, 1)
//   C  [N][6]        ch (ext only)
// Everything else a stage needs (58 words: Mh^-1, kg, T^-1, I_w, r, ubar', contact bits) stays in the
// workspace in global memory (L2-resident) and is streamed by the stage threads every iteration.
struct ArenaLay { int oX, oC, stride; };

constexpr int ITER_MAX_THREADS = 512;  // 16 warps x 128 registers: four warps per SM sub-partition
constexpr int PASS_ENVS = 5;           // envs per pass warp (6 lanes each)
#ifndef PINMPC_ARENA_PAD_MOD
#define PINMPC_ARENA_PAD_MOD 12
#endif
constexpr int ARENA_PAD_MOD = PINMPC_ARENA_PAD_MOD;      // arena stride mod 32 (bank spread of the 6-lane groups)
constexpr int G_MAX = 16;              // envs per CTA
constexpr int CTL_INTS = 32 + 5 * G_MAX;   // done[16] | ndone | pad[15] | red[16][5]

__host__ __device__ inline ArenaLay arena_layout(int N, int ext, int nu)
{
    ArenaLay L;
    L.oX = 72 * N;
    L.oC = L.oX + 8 * N;
    int size = (L.oC + (ext ? 6 * N : 0) + 8 + 3) & ~3;    // + 8: the forward pass reads up to two stages past the horizon
    L.stride = size + ((ARENA_PAD_MOD - (size & 31)) & 31);
    return L;
}

// shared-memory accesses with 32-bit addresses and immediate byte offsets
template <int OFF> __device__ __forceinline__ float lds1(unsigned a)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(v) : "r"(a), "n"(OFF) : "memory");
    return v;
}
template <int OFF> __device__ __forceinline__ float2 lds2(unsigned a)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0,%1}, [%2+%3];" : "=f"(v.x), "=f"(v.y) : "r"(a), "n"(OFF) : "memory");
    return v;
}
template <int OFF> __device__ __forceinline__ float4 lds4(unsigned a)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4+%5];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a), "n"(OFF) : "memory");
    return v;
}
template <int OFF> __device__ __forceinline__ void sts1(unsigned a, float v)
{
    asm volatile("st.shared.f32 [%0+%1], %2;" ::"r"(a), "n"(OFF), "f"(v) : "memory");
}

// word of component i inside the 8-word exchange record  [v0 v1 cos sin v2 v3 v4 v5]
__host__ __device__ constexpr int xslot(int i) { return i < 2 ? i : i + 2; }

// lane-constant description of a pass lane (lane = 6 e + i)
struct PassLane {
    unsigned aK_b, aK_f;     // Kn pair [.][i] (backward), Kn row i (forward), stage 0
    unsigned aXr, aXo, aXq;  // X record of stage 0: base, own slot, the quad holding the own slot
    unsigned aC;             // ch[.][i] (ext)
    int src[6];              // lanes of the env's group
    int nb;                  // lane holding the other component of the (roll, pitch) pair
    int q;                   // own component inside the quad
    float m, om, sg;         // i < 2 ? 1 : 0 ;  1 - m ;  -1, +1, 0 for i = 0, 1, >= 2
    bool act;
};

constexpr int SB_K = 72 * 4, SB_X = 8 * 4, SB_C = 6 * 4;   // bytes per stage of the arena sections

// ---- backward vector pass (the part of the costate driven by sigma0; the response to q and s is
// iteration-invariant and folded into kg by the factorisation).  Lane (e, i) owns component i of
// the (Theta, p) part pq and of the (omega, v) part pv.  Per stage k = N-1..0:
//   hh = sigma0_k + pv -> X_k ;  pq <- pq - Kq^T hh ;  pv <- pv + dt rot(pq) - Kv^T hh
// Instruction order inside a step: the exchange shuffles of the dependent chain go first, the
// operand loads of the next stage are issued in their shadow.
struct BwdOps { float2 k[6]; float4 xq; };

template <int D> __device__ __forceinline__ void bwd_load(BwdOps &o, unsigned aK, unsigned aXq)
{
    o.k[0] = lds2<D * SB_K + 0 * 48>(aK); o.k[1] = lds2<D * SB_K + 1 * 48>(aK); o.k[2] = lds2<D * SB_K + 2 * 48>(aK);
    o.k[3] = lds2<D * SB_K + 3 * 48>(aK); o.k[4] = lds2<D * SB_K + 4 * 48>(aK); o.k[5] = lds2<D * SB_K + 5 * 48>(aK);
    o.xq = lds4<D * SB_X>(aXq);
}

template <int D, bool NEXT>
__device__ __forceinline__ void bwd_step(const BwdOps &o, BwdOps &nxt, float &pq, float &pv, const PassLane &p, unsigned aK, unsigned aXq,
                                         unsigned aXo, float dt)
{
    const float s0 = p.q == 0 ? o.xq.x : p.q == 1 ? o.xq.y : p.q == 2 ? o.xq.z : o.xq.w;
    const float hown = s0 + pv;
    float hh[6];
#pragma unroll
    for (int r = 0; r < 6; r++) hh[r] = __shfl_sync(FULL, hown, p.src[r]);
    const float oth = __shfl_sync(FULL, pq, p.nb);
    if (p.act) sts1<D * SB_X>(aXo, hown);
    if (NEXT) bwd_load<D - 1>(nxt, aK, aXq);
    // off the chain: (A^T p)_v = pv + dt (R_z pq_Theta ; pq_p)   (cos, sin ride in the quad of lanes 0, 1)
    const float al = fmaf(p.m, o.xq.z, p.om), be = p.sg * o.xq.w;
    const float basev = fmaf(dt, fmaf(be, oth, al * pq), pv);
    float a0 = fmaf(o.k[0].x, hh[0], pq), a1 = o.k[3].x * hh[3];
    float b0 = fmaf(o.k[0].y, hh[0], basev), b1 = o.k[3].y * hh[3];
    a0 = fmaf(o.k[1].x, hh[1], a0); a1 = fmaf(o.k[4].x, hh[4], a1); b0 = fmaf(o.k[1].y, hh[1], b0); b1 = fmaf(o.k[4].y, hh[4], b1);
    a0 = fmaf(o.k[2].x, hh[2], a0); a1 = fmaf(o.k[5].x, hh[5], a1); b0 = fmaf(o.k[2].y, hh[2], b0); b1 = fmaf(o.k[5].y, hh[5], b1);
    pq = a0 + a1;
    pv = b0 + b1;
}

__device__ __forceinline__ void backward_pass(const PassLane &p, int N, float dt)
{
    unsigned aK = p.aK_b + (N - 1) * SB_K, aXq = p.aXq + (N - 1) * SB_X, aXo = p.aXo + (N - 1) * SB_X;
    float pq = 0.0f, pv = 0.0f;
    BwdOps A, B;
    bwd_load<0>(A, aK, aXq);
    int k = N - 1;
    for (; k >= 2; k -= 2) {
        bwd_step<0, true>(A, B, pq, pv, p, aK, aXq, aXo, dt);
        bwd_step<-1, true>(B, A, pq, pv, p, aK, aXq, aXo, dt);
        aK -= 2 * SB_K; aXq -= 2 * SB_X; aXo -= 2 * SB_X;
    }
    if (k == 1) {
        bwd_step<0, true>(A, B, pq, pv, p, aK, aXq, aXo, dt);
        bwd_step<-1, false>(B, A, pq, pv, p, aK, aXq, aXo, dt);
    } else {
        bwd_step<0, false>(A, B, pq, pv, p, aK, aXq, aXo, dt);
    }
}

// ---- forward rollout.  Every lane of env e holds the whole state (the (Theta, p) part is advanced
// redundantly, the (omega, v) part is exchanged with shuffles); lane i owns row i of Kh and the new
// component 6 + i.  Per stage k = 0..N-1:   w = kappa_k - Kh x -> X_k ;  x+ = A x + E (w + ch)
// Software pipeline: the part of w_{k+1} that does not depend on the new (omega, v) is computed in
// the shadow of the exchange of stage k; operands are loaded two stages ahead (reads may run up
// to two stages past the horizon: still inside the arena, never used).
struct FwdOps { float4 r0, r1, r2; float kap, c; float2 cs; };

template <int D> __device__ __forceinline__ void fwd_load(FwdOps &o, unsigned aK, unsigned aXo, unsigned aXr, unsigned aC, int has_ext, float gdt)
{
    o.r0 = lds4<D * SB_K>(aK); o.r1 = lds4<D * SB_K + 16>(aK); o.r2 = lds4<D * SB_K + 32>(aK);
    o.kap = lds1<D * SB_X>(aXo);
    o.cs = lds2<D * SB_X + 8>(aXr);
    o.c = has_ext ? gdt + lds1<D * SB_C>(aC) : gdt;
}

// t = kappa + (Theta, p) columns of -Kh x
__device__ __forceinline__ float fwd_pre(const FwdOps &o, const float *xa)
{
    float a0 = fmaf(o.r0.x, xa[0], o.kap), a1 = o.r1.z * xa[3];
    a0 = fmaf(o.r0.z, xa[1], a0); a1 = fmaf(o.r2.x, xa[4], a1);
    a0 = fmaf(o.r1.x, xa[2], a0); a1 = fmaf(o.r2.z, xa[5], a1);
    return a0 + a1;
}

template <int D, bool EMIT>
__device__ __forceinline__ void fwd_step(FwdOps &cur, const FwdOps &nxt, float *xa, float *xb, float &own, float &t, const PassLane &p,
                                         unsigned aK, unsigned aXo, unsigned aXr, unsigned aC, int has_ext, float gdt, float dt, int i,
                                         bool wr, float *ox, float x12)
{
    // on the chain: the (omega, v) columns
    float b0 = fmaf(cur.r0.y, xb[0], t), b1 = cur.r1.w * xb[3];
    b0 = fmaf(cur.r0.w, xb[1], b0); b1 = fmaf(cur.r2.y, xb[4], b1);
    b0 = fmaf(cur.r1.y, xb[2], b0); b1 = fmaf(cur.r2.w, xb[5], b1);
    const float w = b0 + b1;
    const float nun = w + (own + cur.c);
    float nb[6];
#pragma unroll
    for (int j = 0; j < 6; j++) nb[j] = __shfl_sync(FULL, nun, p.src[j]);
    if (p.act) sts1<D * SB_X>(aXo, w);
    // Theta+ = Theta + dt R_z^T omega ; p+ = p + dt v   (old omega, v)
    xa[0] = fmaf(dt, fmaf(cur.cs.x, xb[0], cur.cs.y * xb[1]), xa[0]);
    xa[1] = fmaf(dt, fmaf(cur.cs.x, xb[1], -cur.cs.y * xb[0]), xa[1]);
#pragma unroll
    for (int j = 2; j < 6; j++) xa[j] = fmaf(dt, xb[j], xa[j]);
    fwd_load<D + 2>(cur, aK, aXo, aXr, aC, has_ext, gdt);
    t = fwd_pre(nxt, xa);
    own = nun;
#pragma unroll
    for (int j = 0; j < 6; j++) xb[j] = nb[j];
    if (EMIT) {
        if (wr) {
            const float xs = i == 0 ? xa[0] : i == 1 ? xa[1] : i == 2 ? xa[2] : i == 3 ? xa[3] : i == 4 ? xa[4] : xa[5];
            ox[D * NX + i] = xs;
            ox[D * NX + 6 + i] = nun;
            if (i == 0) ox[D * NX + 12] = x12;
        }
    }
}

template <bool EMIT>
__device__ __forceinline__ void forward_pass(const PassLane &p, int N, float dt, int has_ext, int i, const float *x0s, bool wr, float *ox)
{
    unsigned aK = p.aK_f, aXo = p.aXo, aXr = p.aXr, aC = p.aC;
    float xa[6], xb[6];
#pragma unroll
    for (int j = 0; j < 6; j++) { xa[j] = x0s[j]; xb[j] = x0s[6 + j]; }
    const float x12 = x0s[12];
    float own = x0s[6 + i];
    const float gdt = i == 5 ? dt * x12 : 0.0f;
    FwdOps A, B;
    fwd_load<0>(A, aK, aXo, aXr, aC, has_ext, gdt);
    fwd_load<1>(B, aK, aXo, aXr, aC, has_ext, gdt);
    float t = fwd_pre(A, xa);
    int k = 0;
    for (; k + 1 < N; k += 2) {
        fwd_step<0, EMIT>(A, B, xa, xb, own, t, p, aK, aXo, aXr, aC, has_ext, gdt, dt, i, wr, ox, x12);
        fwd_step<1, EMIT>(B, A, xa, xb, own, t, p, aK, aXo, aXr, aC, has_ext, gdt, dt, i, wr, ox, x12);
        aK += 2 * SB_K; aXo += 2 * SB_X; aXr += 2 * SB_X; aC += 2 * SB_C;
        if (EMIT) ox += 2 * NX;
    }
    if (k < N) fwd_step<0, EMIT>(A, B, xa, xb, own, t, p, aK, aXo, aXr, aC, has_ext, gdt, dt, i, wr, ox, x12);
}

// ---- stage work (one thread, one stage): everything that is local to a stage ------------------------
// Each stage thread owns STAGES_PER_THREAD stages of one env and keeps only z, y and G0 = Gh u0 of
// every owned stage in registers; the stage constants (T^-1, I_w, r, ubar', contact bits, Mh^-1, kg:
// 58 words per stage) are streamed from the L2-resident workspace whenever a phase needs them.
constexpr int STAGES_PER_THREAD = 2;

template <int NU> struct StageState { float z[NU], y[NU]; };

template <int NU> struct StageGeom {
    float TI[6], Iw[6], r[3 * (NW + (NU - 12) / 3)], ru[NU];
    int bits;
};

template <int NU> __device__ __forceinline__ void load_geom(const SrbWs &W, long st, long ts, StageGeom<NU> &g)
{
    constexpr int NC = NW + (NU - 12) / 3, RBW = pinmpc_rb_width(NU);
    const float4 *rec = reinterpret_cast<const float4 *>(W.RB) + ts;
    float v[RBW];
#pragma unroll
    for (int c = 0; c < RBW / 4; c++) {
        const float4 q = __ldg(rec + (long)c * st);
        v[4 * c] = q.x; v[4 * c + 1] = q.y; v[4 * c + 2] = q.z; v[4 * c + 3] = q.w;
    }
#pragma unroll
    for (int c = 0; c < 6; c++) { g.TI[c] = v[c]; g.Iw[c] = v[6 + c]; }
#pragma unroll
    for (int c = 0; c < 3 * NC; c++) g.r[c] = v[12 + c];
#pragma unroll
    for (int c = 0; c < NU; c++) g.ru[c] = v[12 + 3 * NC + c];
    g.bits = __float_as_int(v[12 + 3 * NC + NU]);
}

// X_k = sigma0 = D^-1 Lam^-1 G0
template <int NU>
__device__ __forceinline__ void write_sigma0(const SolveParams &P, const StageGeom<NU> &g, const float *G0, float idt, float m_dt, float *myX)
{
    float l0[6], s0[6];
    lam_inv_apply<NU>(P, g.TI, g.r, G0, l0);
    dinv_apply(g.Iw, idt, m_dt, l0, s0);
    *reinterpret_cast<float2 *>(myX) = make_float2(s0[0], s0[1]);
    *reinterpret_cast<float4 *>(myX + 4) = make_float4(s0[2], s0[3], s0[4], s0[5]);
}

// start of a solve: z, y = the start values, u0 from them, sigma0 -> X
template <int NU>
__device__ __forceinline__ void stage_init(const SolveParams &P, const SrbWs &W, long st, long ts, StageState<NU> &S, float idt, float m_dt,
                                           float *myX, const float *z0, const float *y0)
{
    StageGeom<NU> g;
    load_geom<NU>(W, st, ts, g);
#pragma unroll
    for (int j = 0; j < NU; j++) {
        S.z[j] = z0 ? __ldg(z0 + ts * NU + j) : 0.0f;       // warm start (pinmpc_set_warm_start) or cold start
        S.y[j] = y0 ? __ldg(y0 + ts * NU + j) : 0.0f;
    }
    float u0[NU], G0[6];
    stage_u0<NU>(P, g.ru, S.z, S.y, g.r, u0, G0);
    write_sigma0<NU>(P, g, G0, idt, m_dt, myX);
}

// kappa = Mh^-1 hh - kg  (X: hh -> kappa)
__device__ __forceinline__ void stage_kappa(const SrbWs &W, long st, long ts, float *myX)
{
    float Mi[28];
    const float4 *rec = reinterpret_cast<const float4 *>(W.RA) + ts;
#pragma unroll
    for (int c = 0; c < 7; c++) {
        const float4 q = __ldg(rec + (long)c * st);
        Mi[4 * c] = q.x; Mi[4 * c + 1] = q.y; Mi[4 * c + 2] = q.z; Mi[4 * c + 3] = q.w;
    }
    const float2 h0 = *reinterpret_cast<const float2 *>(myX);
    const float4 h1 = *reinterpret_cast<const float4 *>(myX + 4);
    const float h[6] = { h0.x, h0.y, h1.x, h1.y, h1.z, h1.w };
    float kp[6];
    symv6(Mi, h, kp);
    *reinterpret_cast<float2 *>(myX) = make_float2(kp[0] - Mi[21], kp[1] - Mi[22]);
    *reinterpret_cast<float4 *>(myX + 4) = make_float4(kp[2] - Mi[23], kp[3] - Mi[24], kp[4] - Mi[25], kp[5] - Mi[26]);
}

// u from w, projection (S4), dual update (S5), residuals (S6), contact by contact; then G0 and sigma0 of
// the next iteration.  res = running maxima (r_prim, |dz|, |u|, |z|, |y|) of this thread's env.
template <int NU>
__device__ __forceinline__ void stage_update(const SolveParams &P, const SrbWs &W, long st, long ts, StageState<NU> &S, float idt, float m_dt,
                                             float *myX, bool update, bool emit, bool next, float *ou, float *res, bool two_feet)
{
    constexpr int NC = NW + (NU - 12) / 3;
    StageGeom<NU> g;
    load_geom<NU>(W, st, ts, g);
    float G0[6];
    {
        float u0[NU];
        stage_u0<NU>(P, g.ru, S.z, S.y, g.r, u0, G0);       // G0 = Gh u0 of the current z, y
    }
    if (update) {
        const int bits = g.bits;
        float wv[6], dl[6], lam[6];
        {
            const float2 w0 = *reinterpret_cast<const float2 *>(myX);
            const float4 w1 = *reinterpret_cast<const float4 *>(myX + 4);
            wv[0] = w0.x; wv[1] = w0.y; wv[2] = w1.x; wv[3] = w1.y; wv[4] = w1.z; wv[5] = w1.w;
        }
        dinv_apply(g.Iw, idt, m_dt, wv, dl);
#pragma unroll
        for (int a = 0; a < 6; a++) dl[a] -= G0[a];
        lam_inv_apply<NU>(P, g.TI, g.r, dl, lam);
        float Gn[6] = { 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f };
        // The feet: u of both, then ONE exact projection when no thread of the warp has both feet in stance
        // (a swing foot projects to 0): the wrench of the stance foot is selected, projected and scattered.
        float uf[NW][6], zf[NW][6];
#pragma unroll
        for (int i = 0; i < NW; i++) {
            const float rx = g.r[3 * i], ry = g.r[3 * i + 1], rz = g.r[3 * i + 2];
            const float gl[6] = { fmaf(lam[1], rz, fmaf(-lam[2], ry, lam[3])), fmaf(lam[2], rx, fmaf(-lam[0], rz, lam[4])),
                                  fmaf(lam[0], ry, fmaf(-lam[1], rx, lam[5])), lam[0], lam[1], lam[2] };
#pragma unroll
            for (int a = 0; a < 6; a++) {
                const int c = a < 3 ? fcol(i) + a : mcol(i) + a - 3;
                uf[i][a] = fmaf(P.tR[c], gl[a], fmaf(P.rtR[c], S.z[c] - S.y[c], g.ru[c]));
            }
        }
        {
            const bool on0 = bits & 1, on1 = (bits >> 1) & 1;
            float v0[6], v1[6];
#pragma unroll
            for (int a = 0; a < 6; a++) {
                v0[a] = uf[0][a] + S.y[a < 3 ? fcol(0) + a : mcol(0) + a - 3];
                v1[a] = uf[1][a] + S.y[a < 3 ? fcol(1) + a : mcol(1) + a - 3];
            }
            // one projection of the selected foot (foot 1 if it is in stance, else foot 0) and, only when some thread
            // of the warp has both feet in stance (warp-uniform), a second one of foot 0: two inlined copies, not three
            const bool sel = on1;
            float vs[6], zs[6];
#pragma unroll
            for (int a = 0; a < 6; a++) vs[a] = sel ? v1[a] : v0[a];
            project_wrench(P, vs[0], vs[1], vs[2], vs[3], vs[4], vs[5], zs[0], zs[1], zs[2], zs[3], zs[4], zs[5]);
#pragma unroll
            for (int a = 0; a < 6; a++) { zf[1][a] = on1 ? zs[a] : 0.0f; zf[0][a] = (on0 && !on1) ? zs[a] : 0.0f; }
            if (two_feet) {
                float z0p[6];
                project_wrench(P, v0[0], v0[1], v0[2], v0[3], v0[4], v0[5], z0p[0], z0p[1], z0p[2], z0p[3], z0p[4], z0p[5]);
#pragma unroll
                for (int a = 0; a < 6; a++) zf[0][a] = on0 ? z0p[a] : 0.0f;
            }
        }
#pragma unroll
        for (int i = 0; i < NC; i++) {
            const bool on = (bits >> i) & 1;
            const int fc = fcol(i), mc = mcol(i);
            const float rx = g.r[3 * i], ry = g.r[3 * i + 1], rz = g.r[3 * i + 2];
            constexpr int NV = 6;                           // f (3) and, for a foot, m (3)
            const int nv = i < NW ? 6 : 3;
            int col[NV];
            float ru[NV], uu[NV], zn[NV], u0n[NV];
#pragma unroll
            for (int a = 0; a < NV; a++) ru[a] = 0.0f;
#pragma unroll
            for (int a = 0; a < 3; a++) { col[a] = fc + a; col[3 + a] = mc + a; }
#pragma unroll
            for (int a = 0; a < NV; a++)
                if (a < nv) ru[a] = g.ru[col[a]];
            if (i < NW) {
#pragma unroll
                for (int a = 0; a < 6; a++) { uu[a] = uf[i < NW ? i : 0][a]; zn[a] = zf[i < NW ? i : 0][a]; }
            } else {
                // u = u0 + Rt^-1 Gh^T lam :  f_i += lam_tau x r_i + lam_F
                const float gl[3] = { fmaf(lam[1], rz, fmaf(-lam[2], ry, lam[3])), fmaf(lam[2], rx, fmaf(-lam[0], rz, lam[4])),
                                      fmaf(lam[0], ry, fmaf(-lam[1], rx, lam[5])) };
#pragma unroll
                for (int a = 0; a < 3; a++) {
                    const float u0 = fmaf(P.rtR[col[a]], S.z[col[a]] - S.y[col[a]], ru[a]);
                    uu[a] = fmaf(P.tR[col[a]], gl[a], u0);
                    zn[a] = on ? fminf(fmaxf(uu[a] + S.y[col[a]], -P.hand_fmax), P.hand_fmax) : 0.0f;
                }
            }
#pragma unroll
            for (int a = 0; a < NV; a++)
                if (a < nv) {
                    const float yn = S.y[col[a]] + uu[a] - zn[a];
                    if (emit) {
                        res[0] = fmaxf(res[0], fabsf(uu[a] - zn[a]));
                        res[1] = fmaxf(res[1], fabsf(zn[a] - S.z[col[a]]));
                        res[2] = fmaxf(res[2], fabsf(uu[a])); res[3] = fmaxf(res[3], fabsf(zn[a]));
                        res[4] = fmaxf(res[4], fabsf(yn));
                        ou[col[a]] = uu[a];
                    }
                    S.z[col[a]] = zn[a]; S.y[col[a]] = yn;
                    u0n[a] = fmaf(P.rtR[col[a]], zn[a] - yn, ru[a]);               // u0 of the next iteration
                }
            Gn[0] = fmaf(ry, u0n[2], fmaf(-rz, u0n[1], Gn[0])); Gn[1] = fmaf(rz, u0n[0], fmaf(-rx, u0n[2], Gn[1]));
            Gn[2] = fmaf(rx, u0n[1], fmaf(-ry, u0n[0], Gn[2]));
            Gn[3] += u0n[0]; Gn[4] += u0n[1]; Gn[5] += u0n[2];
            if (i < NW) { Gn[0] += u0n[3]; Gn[1] += u0n[4]; Gn[2] += u0n[5]; }
        }
#pragma unroll
        for (int a = 0; a < 6; a++) G0[a] = Gn[a];
    }
    if (next) write_sigma0<NU>(P, g, G0, idt, m_dt, myX);   // frozen envs keep a well-defined (constant) sigma0
}

template <int NU, bool WARM>
__global__ void __launch_bounds__(ITER_MAX_THREADS) k_iterate_srb(SolveParams P, SrbWs W, const float *__restrict__ x0g,
                                                                  const float *__restrict__ massg, OutPtrs o, int G, int PW, int has_ext, const float *__restrict__ z0g, const float *__restrict__ y0g)
{
    constexpr int NC = NW + (NU - 12) / 3;
    extern __shared__ __align__(16) float smem[];
    const int N = P.N, tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const long st = (long)P.B * N;
    const ArenaLay L = arena_layout(N, has_ext, NU);
    const int b0 = blockIdx.x * G;
    const int Gv = min(G, P.B - b0);
    int *ctl = reinterpret_cast<int *>(smem + G * L.stride);
    int *done = ctl, *ndone = ctl + 16;
    unsigned *red = reinterpret_cast<unsigned *>(ctl + 32);
    float *x0s = smem + G * L.stride + CTL_INTS;          // [G][16] initial states
    const float dt = P.dt, idt = 1.0f / P.dt;

    // ---- load the pass arrays of the CTA's envs into shared memory ------------------------------
    for (int e = 0; e < Gv; e++) {
        float *a = smem + e * L.stride;
        const long s0 = (long)(b0 + e) * N;
        const float4 *src = reinterpret_cast<const float4 *>(W.Kh + s0 * 72);
        float4 *dst = reinterpret_cast<float4 *>(a);
        for (int i = tid; i < N * 18; i += nthr) {
            const float4 v = src[i];
            dst[i] = make_float4(-v.x, -v.y, -v.z, -v.w);
        }
        for (int i = tid; i < N * 2; i += nthr) a[L.oX + (i >> 1) * 8 + 2 + (i & 1)] = W.cs[s0 * 2 + i];
        if (has_ext)
            for (int i = tid; i < N * 6; i += nthr) a[L.oC + i] = W.c6[s0 * 6 + i];
    }
    for (int i = tid; i < CTL_INTS; i += nthr) ctl[i] = 0;
    for (int i = tid; i < Gv * 16; i += nthr) x0s[i] = (i & 15) < NX ? x0g[(long)(b0 + (i >> 4)) * NX + (i & 15)] : 0.0f;

    // ---- pass role of the first PW warps -----------------------------------------------------------
    const bool pass_warp = warp < PW && warp * PASS_ENVS < Gv;   // dedicated: these warps hold no stage state
    PassLane pl;
    int pi = 0, pe = 0;
    {
        const int eloc = lane / 6;
        pi = lane - 6 * eloc;
        const int e = warp * PASS_ENVS + eloc;
        pl.act = pass_warp && eloc < PASS_ENVS && e < Gv;
        // idle lanes shadow the warp's LAST env (the same addresses as its lanes, in the same half-warp: broadcast,
        // no extra shared-memory wavefront)
        const int elast = min(Gv, (warp + 1) * PASS_ENVS) - 1;
        pe = pl.act ? e : (pass_warp ? elast : 0);
        const unsigned ar = (unsigned)__cvta_generic_to_shared(smem + pe * L.stride);
        pl.aK_b = ar + 8 * pi; pl.aK_f = ar + 48 * pi;
        pl.aXr = ar + 4 * L.oX; pl.aXo = pl.aXr + 4 * xslot(pi); pl.aXq = pl.aXr + (pi < 2 ? 0 : 16);
        pl.q = pi < 2 ? pi : pi - 2;
        pl.aC = ar + 4 * (L.oC + pi);
        {
            const int base = pl.act ? 6 * eloc : 6 * (pass_warp ? elast - warp * PASS_ENVS : 0);
#pragma unroll
            for (int r = 0; r < 6; r++) pl.src[r] = base + r;
        }
        pl.nb = lane ^ 1;
        pl.m = pi < 2 ? 1.0f : 0.0f; pl.om = 1.0f - pl.m; pl.sg = pi == 0 ? -1.0f : (pi == 1 ? 1.0f : 0.0f);
        // keep the lane constants in registers: opaque to the compiler, so that it cannot rematerialise them
        // from the lane index inside the pass loops (that costs ~15 instructions per stage of a latency-bound chain)
#pragma unroll
        for (int r = 0; r < 6; r++) asm volatile("" : "+r"(pl.src[r]));
        asm volatile("" : "+r"(pl.nb)); asm volatile("" : "+r"(pl.q));
        asm volatile("" : "+f"(pl.m)); asm volatile("" : "+f"(pl.om)); asm volatile("" : "+f"(pl.sg));
        asm volatile("" : "+r"(pl.aK_b)); asm volatile("" : "+r"(pl.aK_f)); asm volatile("" : "+r"(pl.aXr));
        asm volatile("" : "+r"(pl.aXo)); asm volatile("" : "+r"(pl.aXq)); asm volatile("" : "+r"(pl.aC));
    }
    float *oxe = o.x + (long)(b0 + pe) * N * NX;

    const bool tol_mode = (P.eps_abs > 0.0f || P.eps_rel > 0.0f) && P.check_every > 0;
    if (warp < PW) {
        // =========================== PASS WARP: the sequential recursions, nothing else =============
        for (int it = 0; it < P.iters; it++) {
            const bool is_check = tol_mode && ((it + 1) % P.check_every == 0);
            const bool emit = (it == P.iters - 1) || is_check;
            __syncthreads();                               // X = sigma0 of every stage is in place
            if (pass_warp) backward_pass(pl, N, dt);
            __syncthreads();                               // X = hh
            __syncthreads();                               // X = kappa
            if (pass_warp) {
                if (emit) forward_pass<true>(pl, N, dt, has_ext, pi, x0s + pe * 16, pl.act && !done[pe], oxe);
                else forward_pass<false>(pl, N, dt, has_ext, pi, x0s + pe * 16, false, oxe);
            }
            __syncthreads();                               // X = w
            if (emit) {
                __syncthreads();                           // residuals reduced
                __syncthreads();                           // done flags updated
                if (is_check && *ndone == Gv) break;
            }
        }
        return;
    }

    // ---- STAGE THREADS: thread (env te, slot tj) owns stages tj and tj + H, H = ceil(N / 2) --------------
    const int H = (N + STAGES_PER_THREAD - 1) / STAGES_PER_THREAD;
    const int sid = tid - 32 * PW, nstage = nthr - 32 * PW;
    const int te = sid / H, tj = sid - te * H;
    const bool tact = te < Gv;
    const bool act1 = tact && tj + H < N;                     // the second stage exists
    const int bb = b0 + (tact ? te : 0);
    const long ts0 = (long)bb * N + tj, ts1 = ts0 + (act1 ? H : 0);
    float *arena = smem + (tact ? te : 0) * L.stride;
    float *myX0 = arena + L.oX + tj * 8, *myX1 = myX0 + (act1 ? H * 8 : 0);
    const float m_dt = massg[bb] / dt;

    StageState<NU> S0, S1;
    if (tact) stage_init<NU>(P, W, st, ts0, S0, idt, m_dt, myX0, WARM ? z0g : nullptr, WARM ? y0g : nullptr);
    if (act1) stage_init<NU>(P, W, st, ts1, S1, idt, m_dt, myX1, WARM ? z0g : nullptr, WARM ? y0g : nullptr);
    // does any thread of this warp own a stage with both feet in stance?  (then two projections per stage)
    const bool two_feet0 = __any_sync(FULL, tact && (__float_as_int(__ldg(W.RB + pinmpc_rec_index(12 + 3 * NC + NU, st, ts0))) & 3) == 3);
    const bool two_feet1 = __any_sync(FULL, act1 && (__float_as_int(__ldg(W.RB + pinmpc_rec_index(12 + 3 * NC + NU, st, ts1))) & 3) == 3);
    bool frozen = false;          // this thread's env has met the tolerances (tolerance mode only)

    for (int it = 0; it < P.iters; it++) {
        const bool is_check = tol_mode && ((it + 1) % P.check_every == 0);
        const bool emit = (it == P.iters - 1) || is_check;
        const bool next = it + 1 < P.iters;
        if (emit)
            for (int i = sid; i < 5 * G_MAX; i += nstage) red[i] = 0u;
        __syncthreads();                                   // X = sigma0 of every stage is in place: backward pass
        __syncthreads();                                   // X = hh
        if (tact) stage_kappa(W, st, ts0, myX0);
        if (act1) stage_kappa(W, st, ts1, myX1);
        __syncthreads();                                   // X = kappa: forward pass
        __syncthreads();                                   // X = w
        {
            float res[5] = { 0.0f, 0.0f, 0.0f, 0.0f, 0.0f };
            if (tact) stage_update<NU>(P, W, st, ts0, S0, idt, m_dt, myX0, !frozen, emit, next, o.u + ts0 * NU, res, two_feet0);
            asm volatile("" ::: "memory");              // one stage after the other (register pressure)
            if (act1) stage_update<NU>(P, W, st, ts1, S1, idt, m_dt, myX1, !frozen, emit, next, o.u + ts1 * NU, res, two_feet1);
            if (emit && tact && !frozen) {
                // non-negative floats order like their bit patterns
                atomicMax(&red[te * 5 + 0], __float_as_uint(res[0])); atomicMax(&red[te * 5 + 1], __float_as_uint(res[1]));
                atomicMax(&red[te * 5 + 2], __float_as_uint(res[2])); atomicMax(&red[te * 5 + 3], __float_as_uint(res[3]));
                atomicMax(&red[te * 5 + 4], __float_as_uint(res[4]));
            }
        }
        if (emit) {
            __syncthreads();
            if (sid < Gv && !done[sid]) {                  // one leader per env
                const int e = sid;
                const float rp = __uint_as_float(red[e * 5 + 0]), rd = P.rho * __uint_as_float(red[e * 5 + 1]);
                o.r_prim[b0 + e] = rp; o.r_dual[b0 + e] = rd; o.iters_done[b0 + e] = it + 1;
                if (is_check) {
                    const float sc = fmaxf(__uint_as_float(red[e * 5 + 2]), __uint_as_float(red[e * 5 + 3]));
                    const float ys = __uint_as_float(red[e * 5 + 4]);
                    if (rp <= P.eps_abs + P.eps_rel * sc && rd <= P.eps_abs + P.eps_rel * P.rho * ys) {
                        done[e] = 1;
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
    }
    if (tact) {
        float *oz = o.z + ts0 * NU, *oy = o.y + ts0 * NU;
#pragma unroll
        for (int j = 0; j < NU; j++) { oz[j] = S0.z[j]; oy[j] = S0.y[j]; }
    }
    if (act1) {
        float *oz = o.z + ts1 * NU, *oy = o.y + ts1 * NU;
#pragma unroll
        for (int j = 0; j < NU; j++) { oz[j] = S1.z[j]; oy[j] = S1.y[j]; }
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

size_t iterate_smem_bytes(int N, int G, int ext, int nu)
{
    return ((size_t)G * arena_layout(N, ext, nu).stride + CTL_INTS + 16 * G) * sizeof(float);
}

int iterate_threads(int N, int G)
{
    const int pw = (G + PASS_ENVS - 1) / PASS_ENVS, H = (N + STAGES_PER_THREAD - 1) / STAGES_PER_THREAD;
    return 32 * (pw + (G * H + 31) / 32);
}

// envs per CTA: fewest rounds of the batch over the device first (envs resident per SM, limited by
// shared memory, registers and thread slots), then full pass warps (multiples of PASS_ENVS: a pass
// step costs the same for one env as for five), then the larger CTA (fewer pass warps per SM).
int choose_G(const pinmpc_ctx *h, int regs, int ext)
{
    int best = 0;
    long best_score = 0;
    const int regs_alloc = (regs + 7) / 8 * 8;
    for (int G = 1; G <= G_MAX; G++) {
        const int threads = iterate_threads(h->N, G);
        const size_t smem = iterate_smem_bytes(h->N, G, ext, h->nu);
        if (threads > ITER_MAX_THREADS || smem > (size_t)h->smem_optin) continue;
        int ctas = (int)((size_t)(228 * 1024) / (smem + 1024));
        const int warps_per_smsp = 16384 / (regs_alloc * 32);          // the register file is per sub-partition
        const int by_regs = warps_per_smsp * 4 / (threads / 32), by_thr = 2048 / threads;
        if (by_regs < ctas) ctas = by_regs;
        if (by_thr < ctas) ctas = by_thr;
        if (ctas > 32) ctas = 32;
        if (ctas < 1) continue;
        const long per_round = (long)ctas * G * h->sm_count;
        const long rounds = (h->B + per_round - 1) / per_round;
        const int pw = (G + PASS_ENVS - 1) / PASS_ENVS;
        const long score = -rounds * 1000000 + (G * 1000L) / (pw * PASS_ENVS) * 10 + G;
        if (best == 0 || score > best_score) { best_score = score; best = G; }
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
    const bool prof = h->profiling != 0;
    if (prof) cudaEventRecord(h->ev[0], st);
    k_assemble_srb<NU><<<(unsigned)((stages + 127) / 128), 128, 0, st>>>(P, q, h->srb);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h, "k_assemble_srb launch", e);
    if (prof) cudaEventRecord(h->ev[1], st);
    // which iteration kernel will run is known before the factorisation, which forms the chunk operators of the chunked one
    int tmG = 0, tmC = 0;
    const bool chunked = h->chunks != 1 && (h->chunks > 1 || h->N >= PINMPC_CHUNKED_MIN_N) && pinmpc_tm_config(h, &tmG, &tmC);
    k_factor_srb<<<(unsigned)((h->B + FAC_WARPS * FAC_EPW - 1) / (FAC_WARPS * FAC_EPW)), FAC_WARPS * 32, 0, st>>>(P, q.x0, h->srb, ext,
                                                                                                                chunked ? tmC : 0, h->psi);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h, "k_factor_srb launch", e);
    if (prof) cudaEventRecord(h->ev[2], st);

    // S3-S6: the chunked, TMEM-resident kernel (parallel in the horizon) when the shape fits, else the
    // sequential-pass kernel (also: pinmpc_set_horizon_chunks(h, 1)).  Chosen by measurement (profiles/r2_sweep_config4.md):
    // the chunked kernel wins from N = 20 on (1.05x at N = 20, 1.2x at N = 50, 1.35x at N = 100) and loses below (0.7-0.9x
    // at N = 10, where two chunks of five stages leave nothing to run in parallel).
    int nk = 2;
    if (chunked) {
        const int n = pinmpc_launch_iterate_tm(h, tmG, tmC, st);
        if (n < 0) return -1;
        nk += n;
        h->last_G = tmG; h->last_C = tmC;
    } else {
        // the cold-start kernel carries no warm-start code (same registers and schedule as without the feature)
        auto kern = q.z0 ? k_iterate_srb<NU, true> : k_iterate_srb<NU, false>;
        static std::once_flag fa_once[2];                          // per kernel variant (and per NU: launch_t is a template)
        static cudaFuncAttributes fa_cache[2];
        static cudaError_t fa_err[2];
        const int fi = q.z0 ? 1 : 0;
        std::call_once(fa_once[fi], [&] { fa_err[fi] = cudaFuncGetAttributes(&fa_cache[fi], kern); });
        if (fa_err[fi] != cudaSuccess) return fail(h, "k_iterate_srb attributes", fa_err[fi]);
        const cudaFuncAttributes &fa = fa_cache[fi];
        int G = h->envs_per_cta;
        if (G > G_MAX || (G > 0 && iterate_threads(h->N, G) > ITER_MAX_THREADS) || (G > 0 && iterate_smem_bytes(h->N, G, ext, h->nu) > (size_t)h->smem_optin)) G = 0;
        if (G == 0) G = choose_G(h, fa.numRegs, ext);
        if (G == 0) {
            snprintf(h->err, sizeof h->err, "structured solver: N=%d needs %zu B of shared memory per env (limit %d)", h->N,
                     iterate_smem_bytes(h->N, 1, ext, h->nu), h->smem_optin);
            return -1;
        }
        const int threads = iterate_threads(h->N, G), PW = (G + PASS_ENVS - 1) / PASS_ENVS;
        const size_t smem = iterate_smem_bytes(h->N, G, ext, h->nu);
        // the attributes are process-global per kernel: set once to the device maximum (never per solve, so that handles
        // used from different host threads cannot race between setting and launching)
        static std::once_flag once[2];
        static cudaError_t once_err[2];
        const int wi = q.z0 ? 1 : 0;
        std::call_once(once[wi], [&] {
            once_err[wi] = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, h->smem_optin);
            if (once_err[wi] == cudaSuccess) once_err[wi] = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        });
        if (once_err[wi] != cudaSuccess) return fail(h, "k_iterate_srb smem attribute", once_err[wi]);
        kern<<<(unsigned)((h->B + G - 1) / G), threads, smem, st>>>(P, h->srb, q.x0, q.mass, h->out, G, PW, ext, q.z0, q.y0);
        e = cudaGetLastError();
        if (e != cudaSuccess) return fail(h, "k_iterate_srb launch", e);
        nk += 1;
        h->last_G = G; h->last_C = 1;
    }
    if (prof) { cudaEventRecord(h->ev[3], st); h->prof_valid = true; }
    return nk;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// Test hook of S1 (pinmpc_get_srb_assembly): run the product's assembly kernel and expand ITS records
// (cos sin, I_w, r, ch, mass) back into dense A_k, B_k = E D_k Gh_k, c_k, next to S_k and T_k^-1 as stored.
// ---------------------------------------------------------------------------------------------
namespace {
template <int NU>
__global__ void __launch_bounds__(128) k_srb_expand(SolveParams P, SrbWs W, const float *__restrict__ massg, int has_ext, float *A, float *Bm,
                                                    float *c, float *S, float *Tinv)
{
    constexpr int NC = NW + (NU - 12) / 3;
    const long st = (long)P.B * P.N;
    const long s = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= st) return;
    const int b = (int)(s / P.N);
    const float dt = P.dt, dtm = dt / massg[b];
    float rec[pinmpc_rb_width(NU)];
    for (int w = 0; w < pinmpc_rb_width(NU); w++) rec[w] = W.RB[pinmpc_rec_index(w, st, s)];
    const float Iw[9] = { rec[6], rec[7], rec[8], rec[7], rec[9], rec[10], rec[8], rec[10], rec[11] };
    float Wi[9];
    inv3f(Iw, Wi);
    if (A) {
        float *a = A + s * NX * NX;
        for (int i = 0; i < NX * NX; i++) a[i] = 0.0f;
        for (int i = 0; i < NX; i++) a[i * NX + i] = 1.0f;
        const float cs = W.cs[s * 2], sn = W.cs[s * 2 + 1];
        a[0 * NX + 6] = dt * cs; a[0 * NX + 7] = dt * sn; a[1 * NX + 6] = -dt * sn; a[1 * NX + 7] = dt * cs; a[2 * NX + 8] = dt;   // dt R_z^T
        for (int i = 0; i < 3; i++) a[(3 + i) * NX + 9 + i] = dt;
        a[11 * NX + 12] = dt;
    }
    if (Bm) {
        float *bm = Bm + s * NX * NU;
        for (int i = 0; i < NX * NU; i++) bm[i] = 0.0f;
        for (int i = 0; i < NC; i++) {
            const float rx = rec[12 + 3 * i], ry = rec[13 + 3 * i], rz = rec[14 + 3 * i];
            const float X[9] = { 0.0f, -rz, ry, rz, 0.0f, -rx, -ry, rx, 0.0f };                 // [r]x
            const int fc = fcol(i);
            for (int x = 0; x < 3; x++)
                for (int y = 0; y < 3; y++) {
                    float acc = 0.0f;
                    for (int l = 0; l < 3; l++) acc = fmaf(Wi[x * 3 + l], X[l * 3 + y], acc);
                    bm[(6 + x) * NU + fc + y] = dt * acc;
                    if (i < NW) bm[(6 + x) * NU + mcol(i) + y] = dt * Wi[x * 3 + y];
                }
            for (int x = 0; x < 3; x++) bm[(9 + x) * NU + fc + x] = dtm;
        }
    }
    if (c) {
        float *cc = c + s * NX;
        for (int i = 0; i < NX; i++) cc[i] = 0.0f;
        if (has_ext)
            for (int i = 0; i < 6; i++) cc[6 + i] = W.c6[s * 6 + i];
    }
    if (S)
        for (int i = 0; i < 21; i++) S[s * 21 + i] = W.MI[((long)(i >> 2) * st + s) * 4 + (i & 3)];
    if (Tinv)
        for (int i = 0; i < 6; i++) Tinv[s * 6 + i] = rec[i];
}
}  // namespace

int pinmpc_launch_srb_assembly_debug(pinmpc_ctx *h, float *A, float *Bm, float *c, float *S, float *Tinv, cudaStream_t st)
{
    SolveParams P = make_params(h);
    ProblemPtrs q = make_problem_ptrs(h);
    const long stages = (long)h->B * h->N;
    const unsigned blocks = (unsigned)((stages + 127) / 128);
    const int ext = q.ext != nullptr;
    if (h->nu == 12) {
        k_assemble_srb<12><<<blocks, 128, 0, st>>>(P, q, h->srb);
        k_srb_expand<12><<<blocks, 128, 0, st>>>(P, h->srb, q.mass, ext, A, Bm, c, S, Tinv);
    } else {
        k_assemble_srb<18><<<blocks, 128, 0, st>>>(P, q, h->srb);
        k_srb_expand<18><<<blocks, 128, 0, st>>>(P, h->srb, q.mass, ext, A, Bm, c, S, Tinv);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h, "k_srb_expand launch", e);
    return 2;
}

int pinmpc_launch_solve_srb(pinmpc_ctx *h, cudaStream_t st)
{
    return h->nu == 12 ? launch_t<12>(h, st) : launch_t<18>(h, st);
}
