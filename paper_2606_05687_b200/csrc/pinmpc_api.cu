// pinmpc_api.cu — the C ABI of include/pinmpc.h: argument validation, workspace carving, method
// selection and launch ordering.  Every step of the path runs in the kernels of pinmpc_srb.cu /
// pinmpc_dense.cu; there is no CPU fallback.
#include <new>

#include "pinmpc_common.cuh"

static thread_local char g_create_err[256] = "";

static size_t align_up(size_t v) { return (v + 255) & ~(size_t)255; }

// base workspace: x, u, z, y, r_prim, r_dual, iters_done
size_t pinmpc_ws_base_bytes(int nu, int N, int B)
{
    size_t st = (size_t)B * N;
    return align_up(st * NX * 4) + 3 * align_up(st * nu * 4) + 3 * align_up((size_t)B * 4);
}

// structured-solver factors (SrbWs)
static const int SRB_NARR = 8;
static void srb_sizes(int nu, int N, int B, size_t *f)
{
    size_t st = (size_t)B * N;
    f[0] = st * 72; f[1] = (size_t)B * (N + 1) * 12; f[2] = st * 6; f[3] = st * 2; f[4] = st * 24;
    f[5] = st * PINMPC_RA_W; f[6] = st * (size_t)pinmpc_rb_width(nu);
    f[7] = (size_t)B * pinmpc_psi_cap(N, nu) * 144;
}

size_t pinmpc_ws_srb_bytes(int nu, int N, int B)
{
    size_t f[SRB_NARR], t = 0;
    srb_sizes(nu, N, B, f);
    for (int i = 0; i < SRB_NARR; i++) t += align_up(f[i] * 4);
    return t;
}

// dense extras: A, Bm, c, K, Minv, s, kappa
size_t pinmpc_ws_dense_bytes(int nu, int N, int B)
{
    size_t st = (size_t)B * N;
    return pinmpc_ws_base_bytes(nu, N, B) + pinmpc_ws_srb_bytes(nu, N, B) + align_up(st * NX * NX * 4) + align_up(st * NX * nu * 4) +
           align_up(st * NX * 4) + align_up(st * nu * NX * 4) + align_up(st * nu * nu * 4) + align_up(st * NX * 4) +
           align_up(st * nu * 4);
}

static bool sizes_ok(int nx, int nu, int N, int B, const pinmpc_layout *l, pinmpc_status *why)
{
    if (!l || N < 1 || B < 1) { *why = PINMPC_EINVAL; return false; }
    if (nx != NX || N > PINMPC_N_MAX) { *why = PINMPC_EUNSUPPORTED; return false; }
    if (!(l->n_wrench == 2 && (l->n_force == 0 || l->n_force == 2)) || nu != 6 * l->n_wrench + 3 * l->n_force) {
        *why = PINMPC_EUNSUPPORTED; return false;
    }
    return true;
}

extern "C" size_t pinmpc_workspace_bytes(int nx, int nu, int N, int B, const pinmpc_layout *layout)
{
    pinmpc_status why;
    if (!sizes_ok(nx, nu, N, B, layout, &why)) return 0;
    return pinmpc_ws_base_bytes(nu, N, B) + pinmpc_ws_srb_bytes(nu, N, B);
}

extern "C" size_t pinmpc_workspace_bytes_method(int nx, int nu, int N, int B, const pinmpc_layout *layout, pinmpc_method m)
{
    pinmpc_status why;
    if (!sizes_ok(nx, nu, N, B, layout, &why)) return 0;
    return m == PINMPC_METHOD_DENSE ? pinmpc_ws_dense_bytes(nu, N, B)
                                    : pinmpc_ws_base_bytes(nu, N, B) + pinmpc_ws_srb_bytes(nu, N, B);
}

static pinmpc_status set_err(pinmpc_t h, pinmpc_status s, const char *msg)
{
    if (h) snprintf(h->err, sizeof h->err, "%s", msg);
    else snprintf(g_create_err, sizeof g_create_err, "%s", msg);
    return s;
}

extern "C" pinmpc_status pinmpc_create(pinmpc_t *out, int nx, int nu, int N, int B, const pinmpc_layout *layout,
                                       float rho, int iters, void *d_workspace, size_t workspace_bytes)
{
    if (!out) return set_err(nullptr, PINMPC_EINVAL, "pinmpc_create: out is NULL");
    *out = nullptr;
    pinmpc_status why = PINMPC_OK;
    if (!sizes_ok(nx, nu, N, B, layout, &why))
        return set_err(nullptr, why, "pinmpc_create: unsupported or invalid sizes (nx=13, nu in {12,18}, 1<=N<=512, B>=1)");
    if (!(rho > 0.0f) || iters < 1) return set_err(nullptr, PINMPC_EINVAL, "pinmpc_create: rho must be > 0 and iters >= 1");
    if (!(layout->mu > 0.0f) || !(layout->fz_max > 0.0f) || !(layout->mx_coef > 0.0f) || !(layout->my_coef > 0.0f) ||
        !(layout->mz_coef > 0.0f) || (layout->n_force > 0 && !(layout->hand_fmax >= 0.0f)))
        return set_err(nullptr, PINMPC_EINVAL, "pinmpc_create: layout constants must be positive");
    if (!d_workspace || ((uintptr_t)d_workspace & 255)) return set_err(nullptr, PINMPC_EINVAL, "pinmpc_create: workspace NULL or not 256-byte aligned");
    size_t base = pinmpc_ws_base_bytes(nu, N, B) + pinmpc_ws_srb_bytes(nu, N, B);
    if (workspace_bytes < base) return set_err(nullptr, PINMPC_EALLOC, "pinmpc_create: workspace smaller than pinmpc_workspace_bytes()");

    int dev = 0, major = 0, sms = 0, optin = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) {
        snprintf(g_create_err, sizeof g_create_err, "pinmpc_create: no usable CUDA device: %s", cudaGetErrorString(e));
        return PINMPC_ECUDA;
    }
    if (major != 10) return set_err(nullptr, PINMPC_EUNSUPPORTED, "pinmpc_create: built for sm_100a only (compute capability 10.x required)");

    pinmpc_ctx *h = new (std::nothrow) pinmpc_ctx;
    if (!h) return set_err(nullptr, PINMPC_EALLOC, "pinmpc_create: host allocation failed");
    memset(h, 0, sizeof *h);
    h->nx = nx; h->nu = nu; h->N = N; h->B = B; h->layout = *layout; h->rho = rho; h->iters = iters;
    h->check_every = 1; h->dt = 0.03f; h->method = PINMPC_METHOD_AUTO;
    const float Qdef[NX] = { 500, 500, 100, 50, 50, 200, 1, 1, 1, 20, 20, 10, 0 };
    for (int i = 0; i < NX; i++) h->Qd[i] = Qdef[i];
    for (int i = 0; i < NU_MAX; i++) h->Rd[i] = 1e-5f;
    h->ws = (char *)d_workspace; h->ws_bytes = workspace_bytes; h->sm_count = sms; h->smem_optin = optin;
    h->sticky = cudaSuccess;

    size_t st = (size_t)B * N;
    char *p = h->ws;
    auto take = [&](size_t bytes) { char *r = p; p += align_up(bytes); return r; };
    h->out.x = (float *)take(st * NX * 4);
    h->out.u = (float *)take(st * nu * 4);
    h->out.z = (float *)take(st * nu * 4);
    h->out.y = (float *)take(st * nu * 4);
    h->out.r_prim = (float *)take((size_t)B * 4);
    h->out.r_dual = (float *)take((size_t)B * 4);
    h->out.iters_done = (int *)take((size_t)B * 4);
    {
        size_t f[SRB_NARR];
        srb_sizes(nu, N, B, f);
        h->srb.Kh = (float *)take(f[0] * 4); h->srb.qv = (float *)take(f[1] * 4); h->srb.c6 = (float *)take(f[2] * 4);
        h->srb.cs = (float *)take(f[3] * 4); h->srb.MI = (float *)take(f[4] * 4);
        h->srb.RA = (float *)take(f[5] * 4); h->srb.RB = (float *)take(f[6] * 4);
        h->psi = (float *)take(f[7] * 4); h->psi_cap = pinmpc_psi_cap(N, nu);
    }
    if (workspace_bytes >= pinmpc_ws_dense_bytes(nu, N, B)) {
        h->dA = (float *)take(st * NX * NX * 4);
        h->dB = (float *)take(st * NX * nu * 4);
        h->dC = (float *)take(st * NX * 4);
        h->dK = (float *)take(st * nu * NX * 4);
        h->dMinv = (float *)take(st * nu * nu * 4);
        h->dS = (float *)take(st * NX * 4);
        h->dKappa = (float *)take(st * nu * 4);
    }
    *out = h;
    return PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_set_weights(pinmpc_t h, const float *h_Qdiag, const float *h_Rdiag, float dt)
{
    if (!h) return PINMPC_EINVAL;
    if (!h_Qdiag || !h_Rdiag || !(dt > 0.0f)) return set_err(h, PINMPC_EINVAL, "pinmpc_set_weights: NULL weights or dt <= 0");
    for (int i = 0; i < NX; i++) if (!(h_Qdiag[i] >= 0.0f)) return set_err(h, PINMPC_EINVAL, "pinmpc_set_weights: Q must be >= 0");
    for (int i = 0; i < h->nu; i++) if (!(h_Rdiag[i] >= 0.0f)) return set_err(h, PINMPC_EINVAL, "pinmpc_set_weights: R must be >= 0");
    for (int i = 0; i < NX; i++) h->Qd[i] = h_Qdiag[i];
    for (int i = 0; i < h->nu; i++) h->Rd[i] = h_Rdiag[i];
    h->dt = dt;
    return PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_set_tolerance(pinmpc_t h, float eps_abs, float eps_rel, int check_every)
{
    if (!h) return PINMPC_EINVAL;
    if (!(eps_abs >= 0.0f) || !(eps_rel >= 0.0f) || check_every < 1)
        return set_err(h, PINMPC_EINVAL, "pinmpc_set_tolerance: eps must be >= 0 and check_every >= 1");
    h->eps_abs = eps_abs; h->eps_rel = eps_rel; h->check_every = check_every;
    return PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_set_warm_start(pinmpc_t h, const float *d_z0, const float *d_y0)
{
    if (!h) return PINMPC_EINVAL;
    if ((d_z0 == nullptr) != (d_y0 == nullptr)) return set_err(h, PINMPC_EINVAL, "pinmpc_set_warm_start: give both z0 and y0, or neither");
    h->warm_z = d_z0; h->warm_y = d_y0;
    return PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_set_method(pinmpc_t h, pinmpc_method m)
{
    if (!h) return PINMPC_EINVAL;
    if (m != PINMPC_METHOD_AUTO && m != PINMPC_METHOD_DENSE && m != PINMPC_METHOD_SRB)
        return set_err(h, PINMPC_EINVAL, "pinmpc_set_method: unknown method");
    h->method = m;
    return PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_set_tuning(pinmpc_t h, int envs_per_cta)
{
    if (!h) return PINMPC_EINVAL;
    if (envs_per_cta < 0 || envs_per_cta > 32) return set_err(h, PINMPC_EINVAL, "pinmpc_set_tuning: envs_per_cta must be 0 (auto) .. 32");
    h->envs_per_cta = envs_per_cta;
    return PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_set_horizon_chunks(pinmpc_t h, int chunks)
{
    if (!h) return PINMPC_EINVAL;
    if (chunks < 0 || chunks > h->N) return set_err(h, PINMPC_EINVAL, "pinmpc_set_horizon_chunks: chunks must be 0 (auto), 1 (sequential) .. N");
    if (chunks > 1) {
        pinmpc_ctx t = *h;
        t.chunks = chunks; t.envs_per_cta = 0;
        int G, C;
        if (!pinmpc_tm_config(&t, &G, &C))
            return set_err(h, PINMPC_EUNSUPPORTED, "pinmpc_set_horizon_chunks: needs ceil(N / chunks) <= 6 (4 at nu = 18), chunks <= 128 and chunks <= ceil(N / 5) (ceil(N / 3) at nu = 18)");
    }
    h->chunks = chunks;
    return PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_get_launch_shape(pinmpc_t h, int *envs_per_cta, int *chunks)
{
    if (!h) return PINMPC_EINVAL;
    if (!h->solved) return set_err(h, PINMPC_ESTATE, "pinmpc_get_launch_shape: no solve has been enqueued");
    if (envs_per_cta) *envs_per_cta = h->last_G;
    if (chunks) *chunks = h->last_C;
    return PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_set_problem(pinmpc_t h, const pinmpc_problem *p)
{
    if (!h) return PINMPC_EINVAL;
    if (!p || !p->x0 || !p->x_ref || !p->contact) return set_err(h, PINMPC_EINVAL, "pinmpc_set_problem: x0, x_ref and contact are required");
    h->prob = *p;
    h->have_problem = true;
    h->solved = false;
    return PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_set_dynamics(pinmpc_t h, const float *A, const float *Bm, const float *c)
{
    if (!h) return PINMPC_EINVAL;
    if (!A) { h->have_dynamics = false; h->userA = h->userB = h->userC = nullptr; return PINMPC_OK; }
    if (!Bm) return set_err(h, PINMPC_EINVAL, "pinmpc_set_dynamics: Bm is required with A");
    if (!h->dK) return set_err(h, PINMPC_EALLOC, "pinmpc_set_dynamics: workspace lacks the dense buffers (size it with pinmpc_workspace_bytes_method(..., PINMPC_METHOD_DENSE))");
    h->userA = A; h->userB = Bm; h->userC = c;
    h->have_dynamics = true;
    h->solved = false;
    return PINMPC_OK;
}

static bool raw_inputs_present(const pinmpc_ctx *h)
{
    return h->prob.foot_r && h->prob.yaw && h->prob.mass && h->prob.inertia;
}

extern "C" pinmpc_status pinmpc_solve(pinmpc_t h, void *stream)
{
    if (!h) return PINMPC_EINVAL;
    if (h->sticky != cudaSuccess) return PINMPC_ECUDA;
    if (!h->have_problem) return set_err(h, PINMPC_ESTATE, "pinmpc_solve: call pinmpc_set_problem first");
    cudaStream_t st = (cudaStream_t)stream;
    pinmpc_method m = h->method;
    if (m == PINMPC_METHOD_AUTO) m = h->have_dynamics ? PINMPC_METHOD_DENSE : PINMPC_METHOD_SRB;
    if (m == PINMPC_METHOD_SRB && h->have_dynamics)
        return set_err(h, PINMPC_EINVAL, "pinmpc_solve: the structured solver cannot take pinmpc_set_dynamics matrices");
    if (!h->have_dynamics && !raw_inputs_present(h))
        return set_err(h, PINMPC_EINVAL, "pinmpc_solve: foot_r, yaw, mass and inertia are required without pinmpc_set_dynamics");
    int n;
    if (m == PINMPC_METHOD_DENSE) {
        if (!h->dK) return set_err(h, PINMPC_EALLOC, "pinmpc_solve: workspace lacks the dense buffers");
        n = pinmpc_launch_solve_dense(h, st);
    } else {
        n = pinmpc_launch_solve_srb(h, st);
    }
    if (n < 0) return h->sticky != cudaSuccess ? PINMPC_ECUDA : PINMPC_EUNSUPPORTED;
    h->launch_count = n;
    h->solved = true;
    return PINMPC_OK;
}

static pinmpc_status copy_out(pinmpc_t h, void *dst, const void *src, size_t bytes, cudaStream_t st)
{
    if (!dst) return PINMPC_OK;
    cudaError_t e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, st);
    if (e != cudaSuccess) {
        h->sticky = e;
        snprintf(h->err, sizeof h->err, "cudaMemcpyAsync: %s", cudaGetErrorString(e));
        return PINMPC_ECUDA;
    }
    return PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_get(pinmpc_t h, float *x, float *u, float *r_prim, float *r_dual, int *iters_done, void *stream)
{
    if (!h) return PINMPC_EINVAL;
    if (h->sticky != cudaSuccess) return PINMPC_ECUDA;
    if (!h->solved) return set_err(h, PINMPC_ESTATE, "pinmpc_get: no solve has been enqueued");
    cudaStream_t st = (cudaStream_t)stream;
    size_t n = (size_t)h->B * h->N;
    pinmpc_status s;
    if ((s = copy_out(h, x, h->out.x, n * NX * 4, st))) return s;
    if ((s = copy_out(h, u, h->out.u, n * h->nu * 4, st))) return s;
    if ((s = copy_out(h, r_prim, h->out.r_prim, (size_t)h->B * 4, st))) return s;
    if ((s = copy_out(h, r_dual, h->out.r_dual, (size_t)h->B * 4, st))) return s;
    if ((s = copy_out(h, iters_done, h->out.iters_done, (size_t)h->B * 4, st))) return s;
    return PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_get_aux(pinmpc_t h, float *z, float *y, void *stream)
{
    if (!h) return PINMPC_EINVAL;
    if (h->sticky != cudaSuccess) return PINMPC_ECUDA;
    if (!h->solved) return set_err(h, PINMPC_ESTATE, "pinmpc_get_aux: no solve has been enqueued");
    cudaStream_t st = (cudaStream_t)stream;
    size_t n = (size_t)h->B * h->N * h->nu * 4;
    pinmpc_status s;
    if ((s = copy_out(h, z, h->out.z, n, st))) return s;
    if ((s = copy_out(h, y, h->out.y, n, st))) return s;
    return PINMPC_OK;
}

// receding-horizon shift of the splitting variables: dst[b,k,:] = src[b,min(k+shift,N-1),:]
__global__ void k_shift_stages(const float *__restrict__ src, float *__restrict__ dst, int B, int N, int nu, int shift)
{
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long)B * N * nu) return;
    const int j = (int)(i % nu);
    const long bk = i / nu;
    const int k = (int)(bk % N);
    const long b = bk / N;
    const int ks = min(k + shift, N - 1);
    dst[i] = src[(b * N + ks) * nu + j];
}

extern "C" pinmpc_status pinmpc_shift_aux(pinmpc_t h, int shift, float *z0, float *y0, void *stream)
{
    if (!h) return PINMPC_EINVAL;
    if (h->sticky != cudaSuccess) return PINMPC_ECUDA;
    if (!h->solved) return set_err(h, PINMPC_ESTATE, "pinmpc_shift_aux: no solve has been enqueued");
    if (shift < 0 || shift > h->N || !z0 || !y0) return set_err(h, PINMPC_EINVAL, "pinmpc_shift_aux: 0 <= shift <= N, z0 and y0 non-NULL");
    if (z0 == h->out.z || y0 == h->out.y) return set_err(h, PINMPC_EINVAL, "pinmpc_shift_aux: z0, y0 must not alias the workspace");
    const long n = (long)h->B * h->N * h->nu;
    if (n == 0) return PINMPC_OK;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    k_shift_stages<<<blocks, 256, 0, (cudaStream_t)stream>>>(h->out.z, z0, h->B, h->N, h->nu, shift);
    k_shift_stages<<<blocks, 256, 0, (cudaStream_t)stream>>>(h->out.y, y0, h->B, h->N, h->nu, shift);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { h->sticky = e; return set_err(h, PINMPC_ECUDA, cudaGetErrorString(e)); }
    return PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_get_dynamics(pinmpc_t h, float *A, float *Bm, float *c, void *stream)
{
    if (!h) return PINMPC_EINVAL;
    if (h->sticky != cudaSuccess) return PINMPC_ECUDA;
    if (!h->have_problem || !raw_inputs_present(h)) return set_err(h, PINMPC_ESTATE, "pinmpc_get_dynamics: set_problem with raw inputs first");
    if (!A && !Bm && !c) return PINMPC_OK;
    int n = pinmpc_launch_assemble_dense(h, A, Bm, c, (cudaStream_t)stream);
    return n < 0 ? PINMPC_ECUDA : PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_get_srb_assembly(pinmpc_t h, float *A, float *Bm, float *c, float *S, float *Tinv, void *stream)
{
    if (!h) return PINMPC_EINVAL;
    if (h->sticky != cudaSuccess) return PINMPC_ECUDA;
    if (!h->have_problem || !raw_inputs_present(h)) return set_err(h, PINMPC_ESTATE, "pinmpc_get_srb_assembly: set_problem with raw inputs first");
    int n = pinmpc_launch_srb_assembly_debug(h, A, Bm, c, S, Tinv, (cudaStream_t)stream);
    return n < 0 ? PINMPC_ECUDA : PINMPC_OK;
}

extern "C" int pinmpc_last_launch_count(pinmpc_t h) { return h ? h->launch_count : 0; }

extern "C" pinmpc_status pinmpc_set_profiling(pinmpc_t h, int on)
{
    if (!h) return PINMPC_EINVAL;
    if (on && !h->ev[0]) {
        for (int i = 0; i < 4; i++) {
            cudaError_t e = cudaEventCreate(&h->ev[i]);
            if (e != cudaSuccess) {
                snprintf(h->err, sizeof h->err, "cudaEventCreate: %s", cudaGetErrorString(e));
                return PINMPC_ECUDA;
            }
        }
    }
    h->profiling = on ? 1 : 0;
    h->prof_valid = false;
    return PINMPC_OK;
}

extern "C" pinmpc_status pinmpc_get_kernel_ms(pinmpc_t h, float *h_ms)
{
    if (!h || !h_ms) return PINMPC_EINVAL;
    if (!h->profiling || !h->prof_valid) return set_err(h, PINMPC_ESTATE, "pinmpc_get_kernel_ms: no profiled structured solve");
    cudaError_t e = cudaEventSynchronize(h->ev[3]);
    for (int i = 0; i < 3 && e == cudaSuccess; i++) e = cudaEventElapsedTime(&h_ms[i], h->ev[i], h->ev[i + 1]);
    if (e != cudaSuccess) {
        snprintf(h->err, sizeof h->err, "pinmpc_get_kernel_ms: %s", cudaGetErrorString(e));
        return PINMPC_ECUDA;
    }
    return PINMPC_OK;
}

// Error text of a handle-less entry point (pinmpc_split_solve_static): this thread's handle-less error string.
void pinmpc_note_error(const char *msg) { snprintf(g_create_err, sizeof g_create_err, "%s", msg); }

extern "C" const char *pinmpc_last_error(pinmpc_t h) { return h ? h->err : g_create_err; }

extern "C" void pinmpc_destroy(pinmpc_t h)
{
    if (!h) return;
    for (int i = 0; i < 4; i++)
        if (h->ev[i]) cudaEventDestroy(h->ev[i]);
    delete h;
}
