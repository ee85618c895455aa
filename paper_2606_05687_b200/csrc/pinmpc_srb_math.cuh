// pinmpc_srb_math.cuh — small device helpers of the structured (SRB) formulation shared by the kernels of
// pinmpc_srb.cu (assembly, factorisation, sequential-pass iteration) and pinmpc_tmem.cu (chunked, TMEM-resident
// iteration).  CUDA path only; nothing here is shared with oracle/.
#pragma once
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

// u0 = Rt^-1 (R ubar + rho (z - y)) and its net wrench G0 = Gh u0 for one stage (thread-local);
// ru = Rt^-1 R ubar
template <int NU>
__device__ __forceinline__ void stage_u0(const SolveParams &P, const float *ru, const float *z, const float *y,
                                         const float *r, float *u0, float *G0)
{
    constexpr int NC = NW + (NU - 12) / 3;
#pragma unroll
    for (int j = 0; j < NU; j++) u0[j] = fmaf(P.rtR[j], z[j] - y[j], ru[j]);
#pragma unroll
    for (int a = 0; a < 6; a++) G0[a] = 0.0f;
#pragma unroll
    for (int i = 0; i < NC; i++) {
        const float *f = u0 + fcol(i);
        float rx = r[3 * i], ry = r[3 * i + 1], rz = r[3 * i + 2];
        G0[0] = fmaf(ry, f[2], fmaf(-rz, f[1], G0[0]));
        G0[1] = fmaf(rz, f[0], fmaf(-rx, f[2], G0[1]));
        G0[2] = fmaf(rx, f[1], fmaf(-ry, f[0], G0[2]));
        G0[3] += f[0]; G0[4] += f[1]; G0[5] += f[2];
        if (i < NW) {
            const float *m = u0 + mcol(i);
            G0[0] += m[0]; G0[1] += m[1]; G0[2] += m[2];
        }
    }
}

// y = Lam^-1 x through the Schur complement of the force block:
//   y_t = T^-1 (x_t - C Phi^-1 x_F),  y_F = Phi^-1 (x_F - C^T y_t),
//   C v = sum_i r_i x (t_fi o v),  C^T v = sum_i t_fi o (v x r_i),  Phi = diag(sum_i t_fi)
template <int NU>
__device__ __forceinline__ void lam_inv_apply(const SolveParams &P, const float *TI, const float *r, const float *x, float *y)
{
    constexpr int NC = NW + (NU - 12) / 3;
    const float q0 = P.phi_inv[0] * x[3], q1 = P.phi_inv[1] * x[4], q2 = P.phi_inv[2] * x[5];
    float e0 = x[0], e1 = x[1], e2 = x[2];
#pragma unroll
    for (int i = 0; i < NC; i++) {
        const float rx = r[3 * i], ry = r[3 * i + 1], rz = r[3 * i + 2];
        const float v0 = P.tR[fcol(i)] * q0, v1 = P.tR[fcol(i) + 1] * q1, v2 = P.tR[fcol(i) + 2] * q2;
        e0 = fmaf(rz, v1, fmaf(-ry, v2, e0)); e1 = fmaf(rx, v2, fmaf(-rz, v0, e1)); e2 = fmaf(ry, v0, fmaf(-rx, v1, e2));
    }
    const float t0 = fmaf(TI[0], e0, fmaf(TI[1], e1, TI[2] * e2));
    const float t1 = fmaf(TI[1], e0, fmaf(TI[3], e1, TI[4] * e2));
    const float t2 = fmaf(TI[2], e0, fmaf(TI[4], e1, TI[5] * e2));
    float f0 = x[3], f1 = x[4], f2 = x[5];
#pragma unroll
    for (int i = 0; i < NC; i++) {
        const float rx = r[3 * i], ry = r[3 * i + 1], rz = r[3 * i + 2];
        f0 -= P.tR[fcol(i)] * (t1 * rz - t2 * ry);
        f1 -= P.tR[fcol(i) + 1] * (t2 * rx - t0 * rz);
        f2 -= P.tR[fcol(i) + 2] * (t0 * ry - t1 * rx);
    }
    y[0] = t0; y[1] = t1; y[2] = t2;
    y[3] = P.phi_inv[0] * f0; y[4] = P.phi_inv[1] * f1; y[5] = P.phi_inv[2] * f2;
}

}  // namespace
