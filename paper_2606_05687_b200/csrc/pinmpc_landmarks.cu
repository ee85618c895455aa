// Predictive landmarks and the prediction-confidence reward, eq. (10)-(14).
// Tiny HBM-bound kernels that run after the solve on its stream: the landmarks are gathered straight from
// the solver's x output, nothing goes through the host.
//
// Ring layout (caller-owned, device):  float4 ring[B][NL][N+1] = (c_x, c_y, c_z, target time as int bits),
// slot = target time mod (N+1).  A solve at time t writes target times t+1..t+N only, a reward at time t reads
// target time t only, so a slot is never overwritten before it is read; the stored target time tells a live
// landmark from an old or never-written one (reset writes -1).
#include <cmath>
#include <cstdint>

#include "pinmpc_common.cuh"

namespace {

struct LmParams {
    int B, N, NL;
    int n[PINMPC_MAX_LANDMARKS];         // eq. (10)
    float w[PINMPC_MAX_LANDMARKS][3];    // alpha_l Qc_j / sigma_c^2
};

__global__ void k_landmark_reset(float4 *ring, LmParams p, const uint8_t *mask)
{
    const long per_env = (long)p.NL * (p.N + 1);
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long)p.B * per_env) return;
    if (mask && !mask[i / per_env]) return;
    ring[i] = make_float4(0.0f, 0.0f, 0.0f, __int_as_float(-1));
}

// one thread per (env, landmark): eq. (11)
__global__ void k_landmark_push(float4 *ring, LmParams p, const float *__restrict__ x, const int *__restrict__ t)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.B * p.NL) return;
    const int b = i / p.NL, l = i - b * p.NL;
    const int n = p.n[l], target = t[b] + n;
    const float *c = x + ((long)b * p.N + (n - 1)) * NX + 3;
    int slot = target % (p.N + 1);
    if (slot < 0) slot += p.N + 1;
    ring[((long)b * p.NL + l) * (p.N + 1) + slot] = make_float4(c[0], c[1], c[2], __int_as_float(target));
}

// one thread per env: eq. (12)-(13)
__global__ void k_landmark_reward(const float4 *__restrict__ ring, LmParams p, const float *__restrict__ c_real, const int *__restrict__ t,
                                  float *r, int *n_used)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= p.B) return;
    const int tb = t[b];
    int slot = tb % (p.N + 1);
    if (slot < 0) slot += p.N + 1;
    const float c0 = c_real[b * 3], c1 = c_real[b * 3 + 1], c2 = c_real[b * 3 + 2];
    float acc = 0.0f;
    int used = 0;
    for (int l = 0; l < p.NL; l++) {
        const float4 v = ring[((long)b * p.NL + l) * (p.N + 1) + slot];
        if (__float_as_int(v.w) != tb) continue;          // never stored, or stored for another time
        const float e0 = c0 - v.x, e1 = c1 - v.y, e2 = c2 - v.z;
        acc = fmaf(p.w[l][0], e0 * e0, fmaf(p.w[l][1], e1 * e1, fmaf(p.w[l][2], e2 * e2, acc)));
        used++;
    }
    r[b] = expf(-acc);
    if (n_used) n_used[b] = used;
}

bool make_lm(LmParams &p, int B, int N, const pinmpc_landmark_cfg *cfg)
{
    if (!cfg || B < 0 || N < 1 || cfg->n_landmarks < 1 || cfg->n_landmarks > PINMPC_MAX_LANDMARKS || !(cfg->sigma_c > 0.0f)) return false;
    p.B = B; p.N = N; p.NL = cfg->n_landmarks;
    const double is2 = 1.0 / ((double)cfg->sigma_c * (double)cfg->sigma_c);
    for (int l = 0; l < p.NL; l++) {
        if (!(cfg->s[l] >= 0.0f && cfg->s[l] <= 1.0f)) return false;
        p.n[l] = 1 + (int)std::floor((double)cfg->s[l] * (double)(N - 1));
        for (int j = 0; j < 3; j++) p.w[l][j] = (float)((double)cfg->alpha[l] * (double)cfg->Qc[j] * is2);
    }
    return true;
}

pinmpc_status finish() { return cudaGetLastError() == cudaSuccess ? PINMPC_OK : PINMPC_ECUDA; }

}   // namespace

extern "C" {

size_t pinmpc_landmark_ring_bytes(int B, int N, const pinmpc_landmark_cfg *cfg)
{
    LmParams p;
    if (!make_lm(p, B, N, cfg)) return 0;
    return (size_t)B * p.NL * (N + 1) * sizeof(float4);
}

pinmpc_status pinmpc_landmark_reset(void *d_ring, int B, int N, const pinmpc_landmark_cfg *cfg, const uint8_t *mask, void *stream)
{
    LmParams p;
    if (!make_lm(p, B, N, cfg) || (!d_ring && B > 0)) return PINMPC_EINVAL;
    const long n = (long)B * p.NL * (N + 1);
    if (n == 0) return PINMPC_OK;
    k_landmark_reset<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>((float4 *)d_ring, p, mask);
    return finish();
}

pinmpc_status pinmpc_landmark_push(void *d_ring, int B, int N, const pinmpc_landmark_cfg *cfg, const float *x, const int *t, void *stream)
{
    LmParams p;
    if (!make_lm(p, B, N, cfg) || (B > 0 && (!d_ring || !x || !t))) return PINMPC_EINVAL;
    if (B == 0) return PINMPC_OK;
    k_landmark_push<<<(unsigned)((B * p.NL + 127) / 128), 128, 0, (cudaStream_t)stream>>>((float4 *)d_ring, p, x, t);
    return finish();
}

pinmpc_status pinmpc_landmark_push_solver(pinmpc_t h, void *d_ring, const pinmpc_landmark_cfg *cfg, const int *t, void *stream)
{
    if (!h) return PINMPC_EINVAL;
    if (!h->solved) return PINMPC_ESTATE;
    return pinmpc_landmark_push(d_ring, h->B, h->N, cfg, h->out.x, t, stream);
}

pinmpc_status pinmpc_landmark_reward(const void *d_ring, int B, int N, const pinmpc_landmark_cfg *cfg, const float *c_real, const int *t,
                                     float *r, int *n_used, void *stream)
{
    LmParams p;
    if (!make_lm(p, B, N, cfg) || (B > 0 && (!d_ring || !c_real || !t || !r))) return PINMPC_EINVAL;
    if (B == 0) return PINMPC_OK;
    k_landmark_reward<<<(unsigned)((B + 127) / 128), 128, 0, (cudaStream_t)stream>>>((const float4 *)d_ring, p, c_real, t, r, n_used);
    return finish();
}

}   // extern "C"
