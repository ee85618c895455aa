// pinmpc_dense.cu — the DENSE variant (PINMPC_METHOD_DENSE): generic LTV matrices A_k,B_k,c_k are
// materialised in HBM, the Riccati factors K_k, M_k^{-1}, s_k are computed once per solve and
// streamed from HBM/L2 in every ADMM iteration.  It is the in-house baseline the structured on-chip
// solver (pinmpc_srb.cu) is measured against, and the path behind pinmpc_set_dynamics (arbitrary
// dense A_k,B_k) and pinmpc_get_dynamics.  One warp per env.
//
// Steps (eq. (16)-(17), block order of eq. (21a)-(21c), L186):
//   S1 k_assemble_dense   A_k,B_k,c_k from yaw, contact offsets, mass, inertia (eq. (2)-(4) SRB form)
//   S2 k_factor_dense     P_N = Q; M = Rt + B^T P B; K = M^-1 B^T P A; P = Q + A^T P (A - B K); s = P c
//   S3 k_iterate_dense    backward  g = p - s; h = r + B^T g; kappa = M^-1 h; p = q + A^T g - K^T h
//                         forward   u = -K x + kappa; x+ = A x + B u + c
//   S4-S6 (same kernel)   z = Proj(u + y); y += u - z; residual max-reductions; early exit
#include "pinmpc_common.cuh"

// ---------------------------------------------------------------------------------------------
// S1  dense assembly: one thread per (env, stage)
// ---------------------------------------------------------------------------------------------
__global__ void k_assemble_dense(SolveParams P, ProblemPtrs q, float *__restrict__ A, float *__restrict__ Bm,
                                 float *__restrict__ c)
{
    long s = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= (long)P.B * P.N) return;
    int b = (int)(s / P.N);
    const int nu = P.nu, nc = P.nw + P.nf;
    float Ib[9], Ibi[9], W[9];
#pragma unroll
    for (int i = 0; i < 9; i++) Ib[i] = q.inertia[(long)b * 9 + i];
    inv3f(Ib, Ibi);
    float sn, cs;
    sincosf(q.yaw[s], &sn, &cs);
    world_inertia_inv(Ibi, cs, sn, W);
    const float dt = P.dt, dtm = P.dt / q.mass[b];
    if (A) {
        float *Ak = A + s * (NX * NX);
        for (int i = 0; i < NX * NX; i++) Ak[i] = 0.0f;
        for (int i = 0; i < NX; i++) Ak[i * NX + i] = 1.0f;
        // dTheta = R_z^T omega
        Ak[0 * NX + 6] = dt * cs;  Ak[0 * NX + 7] = dt * sn;
        Ak[1 * NX + 6] = -dt * sn; Ak[1 * NX + 7] = dt * cs;
        Ak[2 * NX + 8] = dt;
        Ak[3 * NX + 9] = dt; Ak[4 * NX + 10] = dt; Ak[5 * NX + 11] = dt;
        Ak[11 * NX + 12] = dt;
    }
    if (Bm) {
        float *Bk = Bm + s * (NX * nu);
        for (int i = 0; i < NX * nu; i++) Bk[i] = 0.0f;
        for (int i = 0; i < nc; i++) {
            const float *r = q.foot_r + (s * nc + i) * 3;
            float rx = r[0], ry = r[1], rz = r[2];
            int fcol = (i < P.nw) ? 3 * i : 6 * P.nw + 3 * (i - P.nw);
            for (int a = 0; a < 3; a++) {
                // row a of W [r]x, [r]x = [[0,-rz,ry],[rz,0,-rx],[-ry,rx,0]]
                float w0 = W[a * 3 + 0], w1 = W[a * 3 + 1], w2 = W[a * 3 + 2];
                Bk[(6 + a) * nu + fcol + 0] = dt * (w1 * rz - w2 * ry);
                Bk[(6 + a) * nu + fcol + 1] = dt * (w2 * rx - w0 * rz);
                Bk[(6 + a) * nu + fcol + 2] = dt * (w0 * ry - w1 * rx);
                Bk[(9 + a) * nu + fcol + a] = dtm;
            }
            if (i < P.nw) {
                int mcol = 3 * P.nw + 3 * i;
                for (int a = 0; a < 3; a++)
                    for (int bb = 0; bb < 3; bb++) Bk[(6 + a) * nu + mcol + bb] = dt * W[a * 3 + bb];
            }
        }
    }
    if (c) {
        float *ck = c + s * NX;
        for (int i = 0; i < NX; i++) ck[i] = 0.0f;
        if (q.ext) {
            const float *e = q.ext + s * 6;
            for (int a = 0; a < 3; a++) {
                ck[6 + a] = dt * (W[a * 3 + 0] * e[3] + W[a * 3 + 1] * e[4] + W[a * 3 + 2] * e[5]);
                ck[9 + a] = dtm * e[a];
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// S2  dense Riccati factorisation: one warp per env, matrices staged in shared memory
// ---------------------------------------------------------------------------------------------
template <int NU>
struct FactorSmem {
    float P[NX * NX], A[NX * NX], B[NX * NU], PB[NX * NU], M[NU * NU], Mi[NU * NU], PA[NX * NX], G[NU * NX],
        K[NU * NX], Phi[NX * NX], T[NX * NX], c[NX];
};

template <int NU>
__global__ void __launch_bounds__(128) k_factor_dense(SolveParams P, DensePtrs d)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int b = blockIdx.x * (blockDim.x >> 5) + wib;
    if (b >= P.B) return;
    FactorSmem<NU> &S = reinterpret_cast<FactorSmem<NU> *>(smem_raw)[wib];
    const int N = P.N;

    for (int i = lane; i < NX * NX; i += 32) S.P[i] = (i / NX == i % NX) ? P.Qd[i / NX] : 0.0f;
    __syncwarp();
    for (int k = N - 1; k >= 0; k--) {
        const long s = (long)b * N + k;
        for (int i = lane; i < NX * NX; i += 32) S.A[i] = d.A[s * (NX * NX) + i];
        for (int i = lane; i < NX * NU; i += 32) S.B[i] = d.Bm[s * (NX * NU) + i];
        if (lane < NX) S.c[lane] = d.c ? d.c[s * NX + lane] : 0.0f;
        __syncwarp();
        // PB = P B ; PA = P A ; s_k = P c
        for (int o = lane; o < NX * NU; o += 32) {
            int i = o / NU, j = o % NU;
            float a = 0.0f;
#pragma unroll
            for (int l = 0; l < NX; l++) a = fmaf(S.P[i * NX + l], S.B[l * NU + j], a);
            S.PB[o] = a;
        }
        for (int o = lane; o < NX * NX; o += 32) {
            int i = o / NX, j = o % NX;
            float a = 0.0f;
#pragma unroll
            for (int l = 0; l < NX; l++) a = fmaf(S.P[i * NX + l], S.A[l * NX + j], a);
            S.PA[o] = a;
        }
        if (lane < NX) {
            float a = 0.0f;
#pragma unroll
            for (int l = 0; l < NX; l++) a = fmaf(S.P[lane * NX + l], S.c[l], a);
            d.s[s * NX + lane] = a;
        }
        __syncwarp();
        // M = Rt + B^T PB ; G = B^T PA
        for (int o = lane; o < NU * NU; o += 32) {
            int i = o / NU, j = o % NU;
            float a = (i == j) ? P.Rd[i] + P.rho : 0.0f;
#pragma unroll
            for (int l = 0; l < NX; l++) a = fmaf(S.B[l * NU + i], S.PB[l * NU + j], a);
            S.M[o] = a;
        }
        for (int o = lane; o < NU * NX; o += 32) {
            int i = o / NX, j = o % NX;
            float a = 0.0f;
#pragma unroll
            for (int l = 0; l < NX; l++) a = fmaf(S.B[l * NU + i], S.PA[l * NX + j], a);
            S.G[o] = a;
        }
        __syncwarp();
        // in-place Cholesky M = L L^T (lower triangle of S.M)
        for (int j = 0; j < NU; j++) {
            if (lane == 0) {
                float dd = S.M[j * NU + j];
                for (int l = 0; l < j; l++) dd = fmaf(-S.M[j * NU + l], S.M[j * NU + l], dd);
                S.M[j * NU + j] = sqrtf(dd);
            }
            __syncwarp();
            if (lane > j && lane < NU) {
                float a = S.M[lane * NU + j];
                for (int l = 0; l < j; l++) a = fmaf(-S.M[lane * NU + l], S.M[j * NU + l], a);
                S.M[lane * NU + j] = a / S.M[j * NU + j];
            }
            __syncwarp();
        }
        // Mi = (L L^T)^{-1}: lane c solves for column c
        if (lane < NU) {
            float t[NU];
#pragma unroll
            for (int i = 0; i < NU; i++) {
                float a = (i == lane) ? 1.0f : 0.0f;
#pragma unroll
                for (int l = 0; l < i; l++) a = fmaf(-S.M[i * NU + l], t[l], a);
                t[i] = a / S.M[i * NU + i];
            }
#pragma unroll
            for (int i = NU - 1; i >= 0; i--) {
                float a = t[i];
#pragma unroll
                for (int l = i + 1; l < NU; l++) a = fmaf(-S.M[l * NU + i], t[l], a);
                t[i] = a / S.M[i * NU + i];
            }
#pragma unroll
            for (int i = 0; i < NU; i++) S.Mi[i * NU + lane] = t[i];
        }
        __syncwarp();
        // K = Mi G
        for (int o = lane; o < NU * NX; o += 32) {
            int i = o / NX, j = o % NX;
            float a = 0.0f;
#pragma unroll
            for (int l = 0; l < NU; l++) a = fmaf(S.Mi[i * NU + l], S.G[l * NX + j], a);
            S.K[o] = a;
        }
        __syncwarp();
        for (int i = lane; i < NU * NX; i += 32) d.K[s * (NU * NX) + i] = S.K[i];
        for (int i = lane; i < NU * NU; i += 32) d.Minv[s * (NU * NU) + i] = S.Mi[i];
        // Phi = A - B K ; T = P Phi ; P = [k>=1] Q + sym(A^T T)
        for (int o = lane; o < NX * NX; o += 32) {
            int i = o / NX, j = o % NX;
            float a = S.A[o];
#pragma unroll
            for (int l = 0; l < NU; l++) a = fmaf(-S.B[i * NU + l], S.K[l * NX + j], a);
            S.Phi[o] = a;
        }
        __syncwarp();
        for (int o = lane; o < NX * NX; o += 32) {
            int i = o / NX, j = o % NX;
            float a = 0.0f;
#pragma unroll
            for (int l = 0; l < NX; l++) a = fmaf(S.P[i * NX + l], S.Phi[l * NX + j], a);
            S.T[o] = a;
        }
        __syncwarp();
        for (int o = lane; o < NX * NX; o += 32) {
            int i = o / NX, j = o % NX;
            float a = 0.0f;
#pragma unroll
            for (int l = 0; l < NX; l++) a = fmaf(S.A[l * NX + i], S.T[l * NX + j], a);
            S.PA[o] = a;   // reuse PA as the unsymmetrised P_k
        }
        __syncwarp();
        for (int o = lane; o < NX * NX; o += 32) {
            int i = o / NX, j = o % NX;
            S.P[o] = 0.5f * (S.PA[i * NX + j] + S.PA[j * NX + i]) + ((k >= 1 && i == j) ? P.Qd[i] : 0.0f);
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------
// S3-S6  dense iteration: one warp per env, lane i owns row i of every vector
// ---------------------------------------------------------------------------------------------
template <int NU>
__global__ void __launch_bounds__(128) k_iterate_dense(SolveParams P, ProblemPtrs q, DensePtrs d, OutPtrs o)
{
    const int lane = threadIdx.x & 31;
    const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (b >= P.B) return;
    const int N = P.N, NW = P.nw;
    const unsigned FULL = 0xffffffffu;
    // which contact does control row `lane` belong to, and which 6 (or 3) rows form its block
    int ci = 0, base_f = 0, base_m = -1, comp = 0;
    if (lane < NU) {
        if (lane < 3 * NW) { ci = lane / 3; comp = lane % 3; base_f = 3 * ci; base_m = 3 * NW + 3 * ci; }
        else if (lane < 6 * NW) { ci = (lane - 3 * NW) / 3; comp = 3 + (lane - 3 * NW) % 3; base_f = 3 * ci; base_m = 3 * NW + 3 * ci; }
        else { ci = NW + (lane - 6 * NW) / 3; comp = (lane - 6 * NW) % 3; base_f = 6 * NW + 3 * (ci - NW); base_m = -1; }
    }
    const int nc = P.nw + P.nf;
    const float Rd_l = (lane < NU) ? P.Rd[lane] : 0.0f;
    const float Qd_l = (lane < NX) ? P.Qd[lane] : 0.0f;
    float *zb = o.z + (long)b * N * NU, *yb = o.y + (long)b * N * NU, *ub = o.u + (long)b * N * NU;
    float *xb = o.x + (long)b * N * NX, *kb = d.kappa + (long)b * N * NU;
    const float *xr = q.x_ref + (long)b * N * NX;
    const float *ur = q.u_ref ? q.u_ref + (long)b * N * NU : nullptr;

    for (int k = 0; k < N; k++)
        if (lane < NU) {
            zb[k * NU + lane] = q.z0 ? q.z0[((long)b * N + k) * NU + lane] : 0.0f;
            yb[k * NU + lane] = q.y0 ? q.y0[((long)b * N + k) * NU + lane] : 0.0f;
        }
    __syncwarp();

    float rp = 0.0f, rd = 0.0f;
    int done = 0;
    for (int it = 0; it < P.iters; it++) {
        // ---- backward vector pass -----------------------------------------------------------
        float p = (lane < NX) ? Qd_l * xr[(N - 1) * NX + lane] : 0.0f;
        for (int k = N - 1; k >= 0; k--) {
            const long s = (long)b * N + k;
            const float *Ak = d.A + s * (NX * NX), *Bk = d.Bm + s * (NX * NU);
            const float *Kk = d.K + s * (NU * NX), *Mk = d.Minv + s * (NU * NU);
            float g = (lane < NX) ? p - d.s[s * NX + lane] : 0.0f;
            float r = 0.0f;
            if (lane < NU) r = Rd_l * (ur ? ur[k * NU + lane] : 0.0f) + P.rho * (zb[k * NU + lane] - yb[k * NU + lane]);
            float h = r;
#pragma unroll
            for (int i = 0; i < NX; i++) {
                float gi = __shfl_sync(FULL, g, i);
                if (lane < NU) h = fmaf(Bk[i * NU + lane], gi, h);
            }
            float kap = 0.0f, pn = (lane < NX && k >= 1) ? Qd_l * xr[(k - 1) * NX + lane] : 0.0f;
#pragma unroll
            for (int l = 0; l < NU; l++) {
                float hl = __shfl_sync(FULL, h, l);
                if (lane < NU) kap = fmaf(Mk[l * NU + lane], hl, kap);      // M^-1 is symmetric
                if (lane < NX) pn = fmaf(-Kk[l * NX + lane], hl, pn);
            }
#pragma unroll
            for (int l = 0; l < NX; l++) {
                float gl = __shfl_sync(FULL, g, l);
                if (lane < NX) pn = fmaf(Ak[l * NX + lane], gl, pn);
            }
            if (lane < NU) kb[k * NU + lane] = kap;
            p = pn;
        }
        // ---- forward rollout + projection + dual update + residuals ---------------------------
        float x = (lane < NX) ? q.x0[(long)b * NX + lane] : 0.0f;
        float un = 0.0f, zn_max = 0.0f, yn = 0.0f;
        rp = 0.0f; rd = 0.0f;
        for (int k = 0; k < N; k++) {
            const long s = (long)b * N + k;
            const float *Ak = d.A + s * (NX * NX), *Bk = d.Bm + s * (NX * NU), *Kk = d.K + s * (NU * NX);
            float u = (lane < NU) ? kb[k * NU + lane] : 0.0f;
            float xn = (lane < NX && d.c) ? d.c[s * NX + lane] : 0.0f;
#pragma unroll
            for (int i = 0; i < NX; i++) {
                float xi = __shfl_sync(FULL, x, i);
                if (lane < NU) u = fmaf(-Kk[lane * NX + i], xi, u);
                if (lane < NX) xn = fmaf(Ak[lane * NX + i], xi, xn);
            }
#pragma unroll
            for (int j = 0; j < NU; j++) {
                float uj = __shfl_sync(FULL, u, j);
                if (lane < NX) xn = fmaf(Bk[lane * NU + j], uj, xn);
            }
            x = xn;
            if (lane < NX) xb[k * NX + lane] = x;
            // projection of v = u + y, every lane gathers the block of its contact
            float yv = (lane < NU) ? yb[k * NU + lane] : 0.0f;
            float zo = (lane < NU) ? zb[k * NU + lane] : 0.0f;
            float v = u + yv;
            float f0 = __shfl_sync(FULL, v, base_f), f1 = __shfl_sync(FULL, v, base_f + 1), f2 = __shfl_sync(FULL, v, base_f + 2);
            int bm = base_m < 0 ? 0 : base_m;
            float m0 = __shfl_sync(FULL, v, bm), m1 = __shfl_sync(FULL, v, bm + 1), m2 = __shfl_sync(FULL, v, bm + 2);
            float zn = 0.0f;
            if (lane < NU) {
                bool on = q.contact[s * nc + ci] != 0;
                if (!on) zn = 0.0f;
                else if (base_m < 0) zn = fminf(fmaxf(v, -P.hand_fmax), P.hand_fmax);
                else {
                    float w[6];
                    project_wrench(P, f0, f1, f2, m0, m1, m2, w[0], w[1], w[2], w[3], w[4], w[5]);
                    zn = comp == 0 ? w[0] : comp == 1 ? w[1] : comp == 2 ? w[2] : comp == 3 ? w[3] : comp == 4 ? w[4] : w[5];
                }
                float ynew = yv + u - zn;
                ub[k * NU + lane] = u; zb[k * NU + lane] = zn; yb[k * NU + lane] = ynew;
                rp = fmaxf(rp, fabsf(u - zn)); rd = fmaxf(rd, fabsf(zn - zo));
                un = fmaxf(un, fabsf(u)); zn_max = fmaxf(zn_max, fabsf(zn)); yn = fmaxf(yn, fabsf(ynew));
            }
        }
        __syncwarp();
        rp = warp_max(rp); rd = P.rho * warp_max(rd);
        done = it + 1;
        if ((P.eps_abs > 0.0f || P.eps_rel > 0.0f) && P.check_every > 0 && done % P.check_every == 0) {
            float sc = fmaxf(warp_max(un), warp_max(zn_max)), ys = warp_max(yn);
            if (rp <= P.eps_abs + P.eps_rel * sc && rd <= P.eps_abs + P.eps_rel * P.rho * ys) break;   // warp-uniform
        }
    }
    if (lane == 0) { o.r_prim[b] = rp; o.r_dual[b] = rd; o.iters_done[b] = done; }
}

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
static int fail(pinmpc_ctx *h, const char *what, cudaError_t e)
{
    h->sticky = e;
    snprintf(h->err, sizeof h->err, "%s: %s", what, cudaGetErrorString(e));
    return -1;
}

int pinmpc_launch_assemble_dense(pinmpc_ctx *h, float *A, float *Bm, float *c, cudaStream_t st)
{
    SolveParams P = make_params(h);
    ProblemPtrs q = make_problem_ptrs(h);
    long n = (long)h->B * h->N;
    k_assemble_dense<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(P, q, A, Bm, c);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h, "k_assemble_dense launch", e);
    return 1;
}

template <int NU>
static int solve_dense_t(pinmpc_ctx *h, cudaStream_t st)
{
    SolveParams P = make_params(h);
    ProblemPtrs q = make_problem_ptrs(h);
    int launches = 0;
    DensePtrs d;
    if (h->have_dynamics) {
        d.A = h->userA; d.Bm = h->userB; d.c = h->userC;
    } else {
        int n = pinmpc_launch_assemble_dense(h, h->dA, h->dB, h->dC, st);
        if (n < 0) return -1;
        launches += n;
        d.A = h->dA; d.Bm = h->dB; d.c = h->dC;
    }
    d.K = h->dK; d.Minv = h->dMinv; d.s = h->dS; d.kappa = h->dKappa;
    const int wpb = 4;
    unsigned grid = (unsigned)((h->B + wpb - 1) / wpb);
    size_t smem = sizeof(FactorSmem<NU>) * wpb;
    cudaError_t e = cudaFuncSetAttribute(k_factor_dense<NU>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return fail(h, "k_factor_dense smem attribute", e);
    k_factor_dense<NU><<<grid, wpb * 32, smem, st>>>(P, d);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h, "k_factor_dense launch", e);
    launches++;
    k_iterate_dense<NU><<<grid, wpb * 32, 0, st>>>(P, q, d, h->out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h, "k_iterate_dense launch", e);
    launches++;
    return launches;
}

int pinmpc_launch_solve_dense(pinmpc_ctx *h, cudaStream_t st)
{
    return h->nu == 12 ? solve_dense_t<12>(h, st) : solve_dense_t<18>(h, st);
}
