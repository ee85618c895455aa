// The paper's own 9-state centroidal model (eq. (1)-(4)): xi = [c ; l_G ; k_G], forward Euler,
//   c+ = c + dt/m l_G,   l_G+ = l_G + dt (m g + sum_i f_i),   k_G+ = k_G + dt sum_i (r_i x f_i + tau_i),
// with the lever r_{i,k} = p_{i,k} - c_k given as data along the linearisation trajectory, i.e. the LTV
// system xi+ = A xi + B_k u + e of eq. (16) with A = [[I, dt/m I, 0],[0, I, 0],[0, 0, I]], e = [0 ; dt m g ; 0] and
// B_k = dt [0 ; I.. ; [r_i]x.. | I..] in the input layout of include/pinmpc.h.  One thread per (stage, row of B).
// The matrices feed the generic LTV entry pinmpc_split_solve_ex with nx = 9.
#include "pinmpc_common.cuh"

namespace {

constexpr int NXC = 9;
constexpr float GRAV = 9.81f;

__global__ void k_assemble_centroidal(int B, int N, int nw, int nf, float dt, const float *__restrict__ mass, const float *__restrict__ foot_r,
                                      float *__restrict__ A, float *__restrict__ Bm, float *__restrict__ e)
{
    const long st = (long)B * N, t = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= st * NXC) return;
    const long s = t / NXC;
    const int row = (int)(t - s * NXC), nc = nw + nf, nu = 6 * nw + 3 * nf;
    const float m = mass[s / N];
    float *Ar = A + (s * NXC + row) * NXC, *Br = Bm + (s * NXC + row) * nu;
    for (int j = 0; j < NXC; j++) Ar[j] = (j == row) ? 1.0f : ((row < 3 && j == row + 3) ? dt / m : 0.0f);
    e[s * NXC + row] = row == 5 ? -dt * m * GRAV : 0.0f;
    for (int j = 0; j < nu; j++) Br[j] = 0.0f;
    if (row < 3) return;
    for (int i = 0; i < nc; i++) {
        const int fc = i < nw ? 3 * i : 6 * nw + 3 * (i - nw);
        if (row < 6) { Br[fc + row - 3] = dt; continue; }                 // l_G rows: dt I for every force
        const float *r = foot_r + (s * nc + i) * 3;                       // k_G rows: dt [r]x for the force, dt I for the moment
        const int a = row - 6;
        // [r]x row a: (0, -r2, r1), (r2, 0, -r0), (-r1, r0, 0)
        Br[fc + (a + 1) % 3] = -dt * r[(a + 2) % 3];
        Br[fc + (a + 2) % 3] = dt * r[(a + 1) % 3];
        if (i < nw) Br[3 * nw + 3 * i + a] = dt;
    }
}

}   // namespace

extern "C" pinmpc_status pinmpc_assemble_centroidal(int B, int N, int n_wrench, int n_force, float dt, const float *mass, const float *foot_r,
                                                    float *A, float *Bm, float *e, void *stream)
{
    if (B < 0 || N < 1 || n_wrench < 0 || n_force < 0 || n_wrench + n_force < 1 || !(dt > 0.0f)) return PINMPC_EINVAL;
    if (B == 0) return PINMPC_OK;
    if (!mass || !foot_r || !A || !Bm || !e) return PINMPC_EINVAL;
    const long tot = (long)B * N * NXC;
    k_assemble_centroidal<<<(unsigned)((tot + 127) / 128), 128, 0, (cudaStream_t)stream>>>(B, N, n_wrench, n_force, dt, mass, foot_r, A, Bm, e);
    return cudaGetLastError() == cudaSuccess ? PINMPC_OK : PINMPC_ECUDA;
}
