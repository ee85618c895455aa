// pinmpc_tmem.cu — the equality step solved IN PARALLEL ACROSS THE HORIZON (north_star (2)
// Remark 2, L23: "horizon-wise recursions" are the bottleneck of GPU MPC), with the gains resident in Blackwell
// TENSOR MEMORY.
//
// The exact LQR step of pinmpc_srb.cu (same formulation, same factors Kh, Mh^-1, kg from k_factor_srb) is a pair
// of affine recursions in the 12-D (Theta, p, omega, v) state,
//     forward   x+ = Phi_k x + E (kappa_k + c_k),           Phi_k = [[I, dt Rot_k], [Kn_a, I + Kn_b]],  Kn = -Kh_k
//     backward  p  <- Phi_k^T p + Kn^T sigma0_k
// The horizon is cut into C chunks of L <= 6 stages.  Each pass is a chunked TWO-SWEEP:
//     sweep A   every chunk concurrently from a zero boundary vector (chunk 0 forward from x_0, the last chunk
//               backward from the zero terminal costate): gives the chunk's affine offset d_c / b_c
//     boundary  x_{k_{c+1}} = Psi_c x_{k_c} + d_c  (backward: p_{k_c} = Psi_c^T p_{k_{c+1}} + b_c), C - 2 dependent
//               12 x 12 steps with the chunk operators Psi_c = Phi_{k_c + L - 1} ... Phi_{k_c} formed once per
//               solve by the factorisation kernel on its backward walk
//     sweep B   every chunk concurrently from its true boundary vector, producing hh -> kappa (backward) and
//               w, x (forward)
// so the dependent depth of a pass drops from N to 2 L + C - 2 (50 -> 19 at N = 50, C = 9).
//
// One CHAIN THREAD per (env, chunk) runs a sweep step alone: 72 FMAs, no shuffles, no shared-memory exchange.
// Its operands, the 72 gains of every stage of its chunk, live in ITS lane of tensor memory (tcgen05.ld
// 32x32b: thread t of warp w reads lane 32 (w % 4) + t; 6 x 72 = 432 of the 512 columns) next to the 6-D
// exchange vector of every stage (sigma0 -> kappa -> w) and the external-wrench offsets.  TMEM is the only
// on-chip store that is both large enough for 14 envs x 50 stages x 72 words (256 KB per SM next to 227 KB of
// shared memory) and fast enough for one-use operands (measured 64 B/clk per sub-partition = 2 x the shared-memory
// pipe of the whole SM); a sweep step is bound by that read rate (144 cycles).  The three WORKER
// threads that share a chain's TMEM lane (warps 4+q, 8+q, 12+q for chain warp q) own two stages of the chunk
// each: u from w, the exact projection (S4), the dual update (S5), residuals (S6) and sigma0 of the next
// iteration, with the stage constants (Mh^-1, kg, T^-1, I_w, r, R ubar) in shared memory — nothing streams from
// L2 after the prologue.
#include <mutex>

#include "pinmpc_srb_math.cuh"

namespace {

#ifndef TM_ABL
#define TM_ABL 0
#endif

constexpr int TM_LMAX = 6;                         // stages per chunk (tensor-memory columns: 6 x 72 gains + exchange + ch)
// stages per chunk actually used: a worker owns half of them with z, y in registers (2 x nu floats per stage), which at
// nu = 18 leaves room for two stages per worker only
__host__ __device__ constexpr int tm_lmax(int nu) { return nu == 12 ? 6 : 4; }
constexpr int TM_XOFF = TM_LMAX * 72;              // exchange vectors   [LMAX][6]   columns 432..467
constexpr int TM_COFF = TM_XOFF + TM_LMAX * 6;     // ch (ext only)      [LMAX][6]   columns 468..503
constexpr int TM_CHAINS = 128;                     // chain threads = TMEM lanes
// worker threads per chain (they share its TMEM lane and split its stages): three at nu = 12 (two stages each, 512 threads
// at 128 registers), two at nu = 18 (384 threads at 168 registers)
__host__ __device__ constexpr int tm_nwpc(int nu) { return nu == 12 ? 3 : 2; }
__host__ __device__ constexpr int tm_threads(int nu) { return 128 * (1 + tm_nwpc(nu)); }
constexpr int TM_GMAX = 32;                        // envs per CTA
constexpr int TM_RAW = 28;                         // Mh^-1 (21) | kg (6) | contact bits
constexpr int TM_CTL = 48 + 5 * TM_GMAX;           // done[32] | ndone | pad[15] | red[32][5]
constexpr unsigned BMASK = 0x00ffffffu;            // the 24 boundary lanes of a worker warp (2 envs x 12 lanes)

__host__ __device__ constexpr int tm_rbw(int nu) { return 12 + 3 * (2 + (nu - 12) / 3) + nu + 2; }   // T^-1 | I_w | r | R ubar' | cos sin

// shared-memory layout (offsets in floats)
struct TmLay { int oA, oB, oPsi, oBnd, oCtl, total; };
__host__ __device__ inline TmLay tm_layout(int N, int G, int C, int nu)
{
    TmLay L;
    const int st = G * N;
    L.oA = 0;
    L.oB = L.oA + TM_RAW * st;
    L.oPsi = L.oB + tm_rbw(nu) * st;
    L.oBnd = L.oPsi + G * (C > 2 ? C - 2 : 0) * 144;
    L.oCtl = L.oBnd + G * (C + 1) * 12;
    L.total = L.oCtl + TM_CTL;
    return L;
}

// ---- tensor memory ------------------------------------------------------------------------------------------
__device__ __forceinline__ void tm_ld8(uint32_t a, float *r)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]), "=f"(r[4]), "=f"(r[5]), "=f"(r[6]), "=f"(r[7]) : "r"(a));
}
__device__ __forceinline__ void tm_ld6(uint32_t a, float *r)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];" : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]) : "r"(a));
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=f"(r[4]), "=f"(r[5]) : "r"(a + 4));
}
__device__ __forceinline__ void tm_st8(uint32_t a, const float *r)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 :: "r"(a), "f"(r[0]), "f"(r[1]), "f"(r[2]), "f"(r[3]), "f"(r[4]), "f"(r[5]), "f"(r[6]), "f"(r[7]) : "memory");
}
__device__ __forceinline__ void tm_st6(uint32_t a, const float *r)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" :: "r"(a), "f"(r[0]), "f"(r[1]), "f"(r[2]), "f"(r[3]) : "memory");
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1,%2};" :: "r"(a + 4), "f"(r[4]), "f"(r[5]) : "memory");
}
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// CTA barrier that also orders tensor-memory stores of one thread before the loads of another
__device__ __forceinline__ void tm_sync()
{
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}

// The chunk operators Psi_c = Phi_{k0+len-1} ... Phi_{k0} of the inner chunks c = 1 .. C-2 (Psi [B][C-2][12][12] row-major) are
// formed by the factorisation kernel on its backward walk (k_factor_srb in pinmpc_srb.cu), once per solve.

// ---------------------------------------------------------------------------------------------
// chain sweeps (one thread = one chunk of one env).  A sweep is software-pipelined over half stages: while
// the 36 gains of one half (three rows of Kn) are consumed, the other half is in flight from tensor memory
// (tcgen05.wait::ld waits for everything outstanding, so exactly one batch is outstanding at a time).
// ---------------------------------------------------------------------------------------------
struct Chain {
    uint32_t tk;          // TMEM address of the chunk's gains (stage j at + 72 j)
    uint32_t sA, sCS;     // shared-memory byte addresses: RA record / (cos, sin) of the chunk's stage 0 (this chain's slot)
    uint32_t jstride;     // bytes from stage j to stage j + 1 of the chunk (slots are stage-major: all chains' stage j together)
    uint32_t xoff;        // extra bytes for the chunk's last stage when it is the one extra stage (compacted slots)
    uint32_t wstride;     // bytes between consecutive float4 groups of a record
    int len;              // stages in the chunk (<= TM_LMAX)
    int nsteps;           // steps of a sweep (warp-uniform): the longest chunk of the CTA
    int base;             // stages every chunk has
};
__device__ __forceinline__ uint32_t chain_joff(const Chain &ch, int j) { return (uint32_t)j * ch.jstride + (j >= ch.base ? ch.xoff : 0u); }

__device__ __forceinline__ float2 lds_f2(uint32_t a)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ float4 lds_f4(uint32_t a)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}

// Packed FP32 pair FMA (sm_100 fma.rn.f32x2): (d0, d1) += (a0, a1) * (b0, b1).  One issue slot for two FMAs; the pairs
// must sit in aligned register pairs, which the callers arrange (consecutive tcgen05.ld destinations, paired states).
__device__ __forceinline__ void ffma2(float &d0, float &d1, float a0, float a1, float b0, float b1)
{
    asm("{ .reg .b64 a, b, c;\n\t mov.b64 a, {%2, %3};\n\t mov.b64 b, {%4, %5};\n\t mov.b64 c, {%0, %1};\n\t fma.rn.f32x2 c, a, b, c;\n\t mov.b64 {%0, %1}, c; }"
        : "+f"(d0), "+f"(d1) : "f"(a0), "f"(a1), "f"(b0), "f"(b1));
}

__device__ __forceinline__ void fadd2(float &d0, float &d1, float a0, float a1, float b0, float b1)      // (d0, d1) = (a0, a1) + (b0, b1)
{
    asm("{ .reg .b64 a, b, c;\n\t mov.b64 a, {%2, %3};\n\t mov.b64 b, {%4, %5};\n\t add.rn.f32x2 c, a, b;\n\t mov.b64 {%0, %1}, c; }"
        : "=f"(d0), "=f"(d1) : "f"(a0), "f"(a1), "f"(b0), "f"(b1));
}

// all 72 gains of stage j of the chunk, row-major Kn[r][0..11]
__device__ __forceinline__ void chain_ld_stage(uint32_t tk, int j, float *k)
{
    const uint32_t a = tk + 72 * j;
#pragma unroll
    for (int q = 0; q < 9; q++) tm_ld8(a + 8 * q, k + 8 * q);
}

// A chunk shorter than the sweep (nsteps) has zero gains, zero exchange vectors and dt, g dt switched off in its unused
// steps, which makes those steps the identity.  Within a step the 72 gains are requested at once and consumed row by
// row as they arrive (the hardware scoreboard tracks every tcgen05.ld destination).

// Backward sweep over the chunk, stages nsteps-1 .. 0:  hh = sigma0 + pv ;  p <- Phi^T p + Kn^T sigma0.
// OUT: kappa = Mh^-1 hh - kg replaces sigma0 in the exchange vector of every stage (an unused step keeps its zero).
// init: the terminal costate (12 floats in shared memory; nullptr = 0); fin: where the costate at the chunk start goes
// (nullptr = nowhere).
template <bool OUT>
__device__ __forceinline__ void chain_bwd_sweep(const Chain &ch, float dt, const float *init, float *fin)
{
    float q[6], v[6];
#pragma unroll
    for (int i = 0; i < 6; i++) { q[i] = init ? init[i] : 0.0f; v[i] = init ? init[6 + i] : 0.0f; }
#pragma unroll 1
    for (int j = ch.nsteps - 1; j >= 0; j--) {
        float k[72], s0[6];
        tm_ld6(ch.tk + TM_XOFF + 6 * j, s0);
        chain_ld_stage(ch.tk, j, k);
        const bool act = j < ch.len;
        const float dte = act ? dt : 0.0f;
        const float2 cs = lds_f2(ch.sCS + chain_joff(ch, j));
#ifndef TM_NOWAIT
        tm_wait_ld();
#endif
        float hh[6];
#pragma unroll
        for (int r = 0; r < 6; r += 2) fadd2(hh[r], hh[r + 1], s0[r], s0[r + 1], v[r], v[r + 1]);
        if (OUT) {
            float Mi[28], kp[6];
            const uint32_t a = ch.sA + chain_joff(ch, j);
#pragma unroll
            for (int c = 0; c < 7; c++) {
                const float4 t = lds_f4(a + c * ch.wstride);
                Mi[4 * c] = t.x; Mi[4 * c + 1] = t.y; Mi[4 * c + 2] = t.z; Mi[4 * c + 3] = t.w;
            }
            symv6(Mi, hh, kp);
#pragma unroll
            for (int r = 0; r < 6; r++) kp[r] = act ? kp[r] - Mi[21 + r] : 0.0f;
            tm_st6(ch.tk + TM_XOFF + 6 * j, kp);
        }
        // (A^T p)_v = pv + dt Rot^T pq  (old pq)
        {
            const float t0 = cs.x * q[0] - cs.y * q[1], t1 = cs.x * q[1] + cs.y * q[0];
            ffma2(v[0], v[1], t0, t1, dte, dte);
#pragma unroll
            for (int i = 2; i < 6; i += 2) ffma2(v[i], v[i + 1], q[i], q[i + 1], dte, dte);
        }
#pragma unroll
        for (int r = 0; r < 6; r++)
#pragma unroll
            for (int i = 0; i < 6; i += 2) {
                ffma2(q[i], q[i + 1], k[12 * r + i], k[12 * r + i + 1], hh[r], hh[r]);
                ffma2(v[i], v[i + 1], k[12 * r + 6 + i], k[12 * r + 7 + i], hh[r], hh[r]);
            }
    }
    if (OUT) tm_wait_st();
    if (fin) {
#pragma unroll
        for (int i = 0; i < 6; i++) { fin[i] = q[i]; fin[6 + i] = v[i]; }
    }
}

// kappa = Mh^-1 hh - kg for every stage of the chunk (hh -> kappa in the exchange vectors; unused steps stay zero)
__device__ __forceinline__ void chain_kappa(const Chain &ch)
{
    tm_wait_st();
    for (int j = 0; j < ch.nsteps; j++) {
        float hh[6], Mi[28], kp[6];
        tm_ld6(ch.tk + TM_XOFF + 6 * j, hh);
        const uint32_t a = ch.sA + chain_joff(ch, j);
#pragma unroll
        for (int c = 0; c < 7; c++) {
            const float4 q = lds_f4(a + c * ch.wstride);
            Mi[4 * c] = q.x; Mi[4 * c + 1] = q.y; Mi[4 * c + 2] = q.z; Mi[4 * c + 3] = q.w;
        }
        tm_wait_ld();
        symv6(Mi, hh, kp);
        const bool act = j < ch.len;
#pragma unroll
        for (int r = 0; r < 6; r++) kp[r] = act ? kp[r] - Mi[21 + r] : 0.0f;
        tm_st6(ch.tk + TM_XOFF + 6 * j, kp);
    }
    tm_wait_st();
}

// Forward sweep over the chunk, stages 0 .. nsteps-1:  w = kappa + Kn x ;  x+ = A x + E (w + c).
// OUT: w replaces kappa in the exchange vector; ox != nullptr (with OUT): x+ -> ox (x_{k+1} of the output).
// init: the start state (12 floats in shared memory; nullptr = 0); fin: where the end state goes (nullptr = nowhere).
template <bool OUT, bool OX = false>
__device__ __forceinline__ void chain_fwd_sweep(const Chain &ch, float dt, float gdt, float x12, int has_ext, const float *init, float *fin, float *ox)
{
    float xa[6], xb[6];
#pragma unroll
    for (int i = 0; i < 6; i++) { xa[i] = init ? init[i] : 0.0f; xb[i] = init ? init[6 + i] : 0.0f; }
#pragma unroll 1
    for (int j = 0; j < ch.nsteps; j++) {
        float k[72], w[6], cv[6];
#pragma unroll
        for (int i = 0; i < 6; i++) cv[i] = 0.0f;
        tm_ld6(ch.tk + TM_XOFF + 6 * j, w);
        if (has_ext) tm_ld6(ch.tk + TM_COFF + 6 * j, cv);
        chain_ld_stage(ch.tk, j, k);
        const bool act = j < ch.len;
        const float dte = act ? dt : 0.0f, gdte = act ? gdt : 0.0f;
        const float2 cs = lds_f2(ch.sCS + chain_joff(ch, j));
#ifndef TM_NOWAIT
        tm_wait_ld();
#endif
#pragma unroll
        for (int r = 0; r < 6; r++) {
            // row r of Kn times (xa ; xb): the products accumulate in one packed sum (even, odd columns); the six rows
            // are independent chains
            float a0 = 0.0f, a1 = 0.0f;
#pragma unroll
            for (int i = 0; i < 6; i += 2) ffma2(a0, a1, k[12 * r + i], k[12 * r + i + 1], xa[i], xa[i + 1]);
#pragma unroll
            for (int i = 0; i < 6; i += 2) ffma2(a0, a1, k[12 * r + 6 + i], k[12 * r + 7 + i], xb[i], xb[i + 1]);
            w[r] += a0 + a1;
        }
        if (OUT) tm_st6(ch.tk + TM_XOFF + 6 * j, w);
        // x_a+ = x_a + dt Rot x_b (old x_b);  x_b+ = x_b + w + c
        {
            const float t0 = fmaf(cs.x, xb[0], cs.y * xb[1]), t1 = fmaf(cs.x, xb[1], -cs.y * xb[0]);
            ffma2(xa[0], xa[1], t0, t1, dte, dte);
#pragma unroll
            for (int i = 2; i < 6; i += 2) ffma2(xa[i], xa[i + 1], xb[i], xb[i + 1], dte, dte);
        }
#pragma unroll
        for (int i = 0; i < 6; i += 2) fadd2(xb[i], xb[i + 1], xb[i], xb[i + 1], w[i], w[i + 1]);
        if (has_ext) {                                      // (uniform)
#pragma unroll
            for (int i = 0; i < 6; i += 2) fadd2(xb[i], xb[i + 1], xb[i], xb[i + 1], cv[i], cv[i + 1]);
        }
        xb[5] += gdte;
        if (OX && ox != nullptr && act) {
            float *o = ox + j * NX;
#pragma unroll
            for (int i = 0; i < 6; i++) { o[i] = xa[i]; o[6 + i] = xb[i]; }
            o[12] = x12;
        }
    }
    if (fin) {
#pragma unroll
        for (int i = 0; i < 6; i++) { fin[i] = xa[i]; fin[6 + i] = xb[i]; }
    }
}

// ---------------------------------------------------------------------------------------------
// stage work of a worker thread (one stage at a time).  Stage records live in shared memory as float4 groups,
// group-major over SLOTS (rec[group][slot], slot = the stage's position in lane order), so that the 32 lanes of a
// warp read consecutive float4s (conflict-free LDS.128).  RB record (words): T^-1 (6) | I_w (6) | r (3 nc) |
// R ubar' (nu) | cos sin.  The groups are (re)loaded phase by phase, so that next to z, y of the owned stages only a
// few dozen registers are live.
// ---------------------------------------------------------------------------------------------
template <int NU> struct TmState { float z[NU], y[NU]; };

#define TM_PHASE() asm volatile("" ::: "memory")
// -DPINMPC_TM_TIMING=2: lane 0 of every worker warp of CTA 0 also stores clock() between the phases of the stage update
#if defined(PINMPC_TM_TIMING) && PINMPC_TM_TIMING >= 2
#define PINMPC_TM_UTIMING
#endif
#ifdef PINMPC_TM_UTIMING
__device__ int g_ut[16 * 32];
#define TM_UT(i) { if (ut != nullptr) { asm volatile("" ::: "memory"); ut[i] = (int)clock(); asm volatile("" ::: "memory"); } }
#define TM_UTARG , int *ut
#else
#define TM_UT(i)
#define TM_UTARG
#endif

// float4 groups [G0, G1) of a record -> v (v[0] = word 4 G0)
template <int G0, int G1>
__device__ __forceinline__ void tm_ld_groups(uint32_t rec, uint32_t gstride, float *v)      // rec: shared-memory byte address of group 0
{
#pragma unroll
    for (int g = G0; g < G1; g++) {
        const float4 q = lds_f4(rec + g * gstride);
        v[4 * (g - G0)] = q.x; v[4 * (g - G0) + 1] = q.y; v[4 * (g - G0) + 2] = q.z; v[4 * (g - G0) + 3] = q.w;
    }
}

// G = Gh u0,  u0 = Rt^-1 (R ubar + rho (z - y));  v = the record from word 12 on (r | R ubar')
template <int NU>
__device__ __forceinline__ void tm_gh_u0(const SolveParams &P, const float *v, const float *z, const float *y, float *G)
{
    constexpr int NC = NW + (NU - 12) / 3;
    const float *rr = v, *ru = v + 3 * NC;
#pragma unroll
    for (int a = 0; a < 6; a++) G[a] = 0.0f;
#pragma unroll
    for (int i = 0; i < NC; i++) {
        const int fc = fcol(i);
        const float rx = rr[3 * i], ry = rr[3 * i + 1], rz = rr[3 * i + 2];
        float f[3];
#pragma unroll
        for (int a = 0; a < 3; a++) f[a] = fmaf(P.rtR[fc + a], z[fc + a] - y[fc + a], ru[fc + a]);
        G[0] = fmaf(ry, f[2], fmaf(-rz, f[1], G[0]));
        G[1] = fmaf(rz, f[0], fmaf(-rx, f[2], G[1]));
        G[2] = fmaf(rx, f[1], fmaf(-ry, f[0], G[2]));
        G[3] += f[0]; G[4] += f[1]; G[5] += f[2];
        if (i < NW) {
            const int mc = mcol(i);
#pragma unroll
            for (int a = 0; a < 3; a++) G[a] += fmaf(P.rtR[mc + a], z[mc + a] - y[mc + a], ru[mc + a]);
        }
    }
}

// sigma0 = D^-1 Lam^-1 G;  geo = the record's words 0 .. 12 + 3 nc (T^-1 | I_w | r)
template <int NU>
__device__ __forceinline__ void tm_sigma0(const SolveParams &P, const float *geo, const float *G, float idt, float m_dt, float *s0)
{
    float l0[6];
    lam_inv_apply<NU>(P, geo, geo + 12, G, l0);
    dinv_apply(geo + 6, idt, m_dt, l0, s0);
}

// u from w, projection (S4), dual update (S5), residuals (S6); then sigma0 of the next iteration.
// wv: in w of this stage, out sigma0 of the next iteration.  res = running maxima (r_prim, |dz|, |u|, |z|, |y|).
template <int NU, bool EMIT>
__device__ __forceinline__ void tm_stage_update(const SolveParams &P, uint32_t rb, uint32_t nsl, int bits, float *z, float *y, float idt, float m_dt,
                                                float *wv, bool update, float *ou, float *res, bool two_feet TM_UTARG)
{
    TM_UT(0)
    constexpr int NC = NW + (NU - 12) / 3, RBW = tm_rbw(NU);
    constexpr int GEO4 = (12 + 3 * NC + 3) / 4;                 // groups holding T^-1, I_w, r
    float G0[6];
    {
        float v[RBW - 12];
        tm_ld_groups<3, RBW / 4>(rb, nsl, v);
        tm_gh_u0<NU>(P, v, z, y, G0);
    }
    TM_PHASE();
    TM_UT(1)
    if (update) {
        float lam[6];
        {
            float geo[4 * GEO4], dl[6];
            tm_ld_groups<0, GEO4>(rb, nsl, geo);
            dinv_apply(geo + 6, idt, m_dt, wv, dl);
#pragma unroll
            for (int a = 0; a < 6; a++) dl[a] -= G0[a];
            lam_inv_apply<NU>(P, geo, geo + 12, dl, lam);
        }
        TM_PHASE();
        TM_UT(2)
        // u = u0 + Rt^-1 Gh^T lam, contact by contact;  y <- y + u  (= the argument v of the projection)
        float uk[EMIT ? NU : 1];
        {
            float v[RBW - 12];
            tm_ld_groups<3, RBW / 4>(rb, nsl, v);
            const float *rr = v, *ru = v + 3 * NC;
#pragma unroll
            for (int i = 0; i < NC; i++) {
                const float rx = rr[3 * i], ry = rr[3 * i + 1], rz = rr[3 * i + 2];
                const float gl[6] = { fmaf(lam[1], rz, fmaf(-lam[2], ry, lam[3])), fmaf(lam[2], rx, fmaf(-lam[0], rz, lam[4])),
                                      fmaf(lam[0], ry, fmaf(-lam[1], rx, lam[5])), lam[0], lam[1], lam[2] };
#pragma unroll
                for (int a = 0; a < (i < NW ? 6 : 3); a++) {
                    const int c = a < 3 ? fcol(i) + a : mcol(i) + a - 3;
                    const float u = fmaf(P.tR[c], gl[a], fmaf(P.rtR[c], z[c] - y[c], ru[c]));
                    if (EMIT) { uk[c] = u; ou[c] = u; res[2] = fmaxf(res[2], fabsf(u)); }
                    y[c] += u;
                }
            }
        }
        TM_PHASE();
        TM_UT(3)
        // the feet: ONE exact projection when no thread of the warp has both feet in stance (a swing foot projects to
        // 0): the argument of the stance foot is selected, projected and scattered; else a second one of foot 0
        float zf[NW][6];
        {
            const bool on0 = bits & 1, on1 = (bits >> 1) & 1;
            float vs[6], zs[6];
#pragma unroll
            for (int a = 0; a < 6; a++) {
                const int c0 = a < 3 ? fcol(0) + a : mcol(0) + a - 3, c1 = a < 3 ? fcol(1) + a : mcol(1) + a - 3;
                vs[a] = on1 ? y[c1] : y[c0];
            }
            project_wrench(P, vs[0], vs[1], vs[2], vs[3], vs[4], vs[5], zs[0], zs[1], zs[2], zs[3], zs[4], zs[5]);
#pragma unroll
            for (int a = 0; a < 6; a++) { zf[1][a] = on1 ? zs[a] : 0.0f; zf[0][a] = (on0 && !on1) ? zs[a] : 0.0f; }
            if (two_feet) {
                float z0p[6];
                project_wrench(P, y[fcol(0)], y[fcol(0) + 1], y[fcol(0) + 2], y[mcol(0)], y[mcol(0) + 1], y[mcol(0) + 2], z0p[0], z0p[1], z0p[2],
                               z0p[3], z0p[4], z0p[5]);
#pragma unroll
                for (int a = 0; a < 6; a++) zf[0][a] = on0 ? z0p[a] : 0.0f;
            }
        }
        TM_UT(4)
        // z <- projection, y <- v - z
#pragma unroll
        for (int i = 0; i < NC; i++) {
            const bool on = (bits >> i) & 1;
#pragma unroll
            for (int a = 0; a < (i < NW ? 6 : 3); a++) {
                const int c = a < 3 ? fcol(i) + a : mcol(i) + a - 3;
                const float zn = i < NW ? zf[i < NW ? i : 0][a] : (on ? fminf(fmaxf(y[c], -P.hand_fmax), P.hand_fmax) : 0.0f);
                const float yn = y[c] - zn;
                if (EMIT) {
                    res[0] = fmaxf(res[0], fabsf(uk[c] - zn));
                    res[1] = fmaxf(res[1], fabsf(zn - z[c]));
                    res[3] = fmaxf(res[3], fabsf(zn)); res[4] = fmaxf(res[4], fabsf(yn));
                }
                z[c] = zn; y[c] = yn;
            }
        }
        TM_PHASE();
        TM_UT(5)
        {
            float v[RBW - 12];
            tm_ld_groups<3, RBW / 4>(rb, nsl, v);
            tm_gh_u0<NU>(P, v, z, y, G0);                       // Gh u0 of the next iteration
        }
        TM_PHASE();
        TM_UT(6)
    }
    {
        float geo[4 * GEO4];
        tm_ld_groups<0, GEO4>(rb, nsl, geo);
        tm_sigma0<NU>(P, geo, G0, idt, m_dt, wv);               // frozen envs keep a well-defined (constant) sigma0
    }
    TM_UT(7)
}

#ifdef PINMPC_TM_TIMING
// timestamps of one iteration (chain: thread 0 -> pad[0..6], worker: thread 128 -> pad[7..13]); read after a barrier-protected load
#define TM_TICK(i) { if (it == TM_TICK_IT && (threadIdx.x == 0 || threadIdx.x == 128)) { int dmy_ = *(volatile int *)ndone; asm volatile("" :: "r"(dmy_) : "memory"); \
                     ((volatile int *)ndone)[1 + (threadIdx.x == 0 ? 0 : 7) + (i)] = (int)clock(); } }
#define TM_TICK_IT 50
#else
#define TM_TICK(i)
#endif

// ---------------------------------------------------------------------------------------------
// The iteration loop of a chain warp.  NOT inlined on purpose: the chain loop then gets its own register
// allocation (operand buffers of a whole stage), independent of the stage-update code of the worker warps in the
// kernel body; a value spilled in a sweep loop would cost an L2 round trip per step (the 227 KB of shared memory
// leave no L1 for local memory).
// ---------------------------------------------------------------------------------------------
struct ChainArgs {
    Chain ch;
    float dt, gdt, x12;
    int has_ext, iters, check_every, tol_mode, C, cc, cvalid, Gv;
    float *slot_lo, *oxe;
    int *done_e, *ndone;
};

template <int RBW>
__device__ __noinline__ void tm_chain_main(ChainArgs A)
{
    Chain ch = A.ch;
    // Warp-uniform by construction; the broadcast from lane 0 tells the compiler, which then keeps the tensor-memory
    // addresses and the loop counters of the sweeps in uniform registers (no R2UR per tcgen05.ld: 6-13 per step before).
    ch.tk = __shfl_sync(FULL, ch.tk, 0);
    ch.nsteps = __shfl_sync(FULL, ch.nsteps, 0);
    const float dt = A.dt, gdt = A.gdt, x12 = A.x12;
    const int has_ext = __shfl_sync(FULL, A.has_ext, 0), C = __shfl_sync(FULL, A.C, 0), cc = A.cc;
    A.iters = __shfl_sync(FULL, A.iters, 0); A.tol_mode = __shfl_sync(FULL, A.tol_mode, 0); A.check_every = __shfl_sync(FULL, A.check_every, 0);
    const bool cvalid = A.cvalid != 0;
    float *slot_lo = A.slot_lo, *slot_hi = A.slot_lo + 12, *oxe = A.oxe;
    int *ndone = A.ndone;
    for (int it = 0; it < A.iters; it++) {
        const bool is_check = A.tol_mode && ((it + 1) % A.check_every == 0);
        const bool emit = __shfl_sync(FULL, (int)((it == A.iters - 1) || is_check), 0) != 0;   // (the modulo hides its uniformity)
        tm_sync();                                          // (1) sigma0 of every stage is in the exchange vectors
        TM_TICK(0)
        // ---- backward sweep A: zero terminal costate -> b_c (the last chunk: its true costate)
        if (C > 1 && TM_ABL != 3 && TM_ABL != 4) chain_bwd_sweep<false>(ch, dt, nullptr, (cvalid && cc >= 1) ? slot_lo : nullptr);
        TM_TICK(1)
        __syncthreads();                                    // (2) boundary recursion (workers)
        __syncthreads();                                    // (3) true terminal costates in the slots
        TM_TICK(2)
        // ---- backward sweep B: true terminal costate; kappa -> exchange
        if (TM_ABL != 4) chain_bwd_sweep<true>(ch, dt, slot_hi, nullptr);
        TM_TICK(3)
        // ---- forward sweep A: zero start state (chunk 0: x_0) -> d_c (chunk 0: its true end state)
        if (C > 1 && TM_ABL != 3 && TM_ABL != 4)
            chain_fwd_sweep<false>(ch, dt, gdt, x12, has_ext, cc == 0 ? slot_lo : nullptr, (cvalid && cc <= C - 2) ? slot_hi : nullptr, nullptr);
        TM_TICK(4)
        __syncthreads();                                    // (4) boundary recursion (workers)
        __syncthreads();                                    // (5) true start states in the slots
        TM_TICK(5)
        // ---- forward sweep B: true start state; w -> exchange, x -> output
        if (TM_ABL != 4) {
            if (emit) chain_fwd_sweep<true, true>(ch, dt, gdt, x12, has_ext, slot_lo, nullptr, (cvalid && !*A.done_e) ? oxe : nullptr);
            else chain_fwd_sweep<true, false>(ch, dt, gdt, x12, has_ext, slot_lo, nullptr, nullptr);     // no state output code in the common step
        }
        TM_TICK(6)
        tm_sync();                                          // (6) w of every stage is in the exchange vectors
        if (emit) {
            __syncthreads();                                // residuals reduced
            __syncthreads();                                // done flags updated
            if (is_check && *ndone == A.Gv) break;
        }
    }
}

// Prologue of a chain thread: the gains of its chunk -> its lane of tensor memory, row-major Kn[r][0..11] = -Kh[r][.]
// (Kh arrives as the pairs (Kh[r][j], Kh[r][6+j])), and the chunk's ch rows.  Its own function: the 36 loads in flight
// per trip must not count against the register allocation of the kernel body.
__device__ __noinline__ void tm_chain_load(const float *__restrict__ Kh, const float *__restrict__ c6, int clen, uint32_t myt)
{
    for (int j0 = 0; j0 < TM_LMAX; j0 += 1) {                      // one stage per trip: 18 loads in flight
        float4 v[1][18];
#pragma unroll
        for (int t = 0; t < 1; t++) {
            const int j = j0 + t;
            const float4 *src = reinterpret_cast<const float4 *>(Kh + (long)(j < clen ? j : 0) * 72);
#pragma unroll
            for (int i = 0; i < 18; i++) v[t][i] = __ldg(src + i);
        }
#pragma unroll
        for (int t = 0; t < 1; t++) {
            const int j = j0 + t;
            const float m = j < clen ? -1.0f : 0.0f;            // Kn = -Kh; zero gains in the unused steps of a short chunk
            float kq[72];
#pragma unroll
            for (int r = 0; r < 6; r++) {
                const float4 v0 = v[t][3 * r], v1 = v[t][3 * r + 1], v2 = v[t][3 * r + 2];
                float *d = kq + 12 * r;
                d[0] = m * v0.x; d[6] = m * v0.y; d[1] = m * v0.z; d[7] = m * v0.w;
                d[2] = m * v1.x; d[8] = m * v1.y; d[3] = m * v1.z; d[9] = m * v1.w;
                d[4] = m * v2.x; d[10] = m * v2.y; d[5] = m * v2.z; d[11] = m * v2.w;
            }
#pragma unroll
            for (int c = 0; c < 9; c++) tm_st8(myt + 72 * j + 8 * c, kq + 8 * c);
            float cv[6] = { 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f };
            if (c6 != nullptr && j < clen) {
#pragma unroll
                for (int i = 0; i < 6; i++) cv[i] = __ldg(c6 + j * 6 + i);
            }
            tm_st6(myt + TM_COFF + 6 * j, cv);
        }
    }
    tm_wait_st();
}

// Prologue of the CTA: stage records of its envs -> shared memory (float4 groups, slot-major), chunk operators,
// boundary slots, control words.  Its own function for the same reason as tm_chain_load.
template <int NU>
__device__ __noinline__ void tm_cta_load(SrbWs W, const float *__restrict__ Psi, const float *__restrict__ x0g, long st, int b0, int Gv, int N, int G,
                                          int C, float *smem)
{
    constexpr int GRBW = pinmpc_rb_width(NU);
    const int tid = threadIdx.x;
    const TmLay L = tm_layout(N, G, C, NU);
    float4 *recA4 = reinterpret_cast<float4 *>(smem + L.oA), *recB4 = reinterpret_cast<float4 *>(smem + L.oB);
    float *psi = smem + L.oPsi, *bnd = smem + L.oBnd;
    int *ctl = reinterpret_cast<int *>(smem + L.oCtl);
    const int nsl = G * N, nch = G * C, cbase = N / C, crem = N - cbase * C, nst = Gv * N;
    const float4 *RA4 = reinterpret_cast<const float4 *>(W.RA), *RB4 = reinterpret_cast<const float4 *>(W.RB);
    const long s0 = (long)b0 * N;
    const int big = crem * (cbase + 1);                          // stages covered by the longer chunks
    constexpr int TM_THREADS = tm_threads(NU);
    for (int sl = tid; sl < nst; sl += TM_THREADS) {              // one stage per thread and trip, all its groups in flight
        const int e = sl / N, k = sl - e * N;
        int c, j;
        if (k < big) { c = k / (cbase + 1); j = k - c * (cbase + 1); }
        else { c = crem + (k - big) / cbase; j = (k - big) - (c - crem) * cbase; }
        const int slot = j < cbase ? j * nch + e * C + c : cbase * nch + e * crem + c;
        float4 va[7], vb[GRBW / 4];
#pragma unroll
        for (int g = 0; g < 7; g++) va[g] = __ldg(RA4 + (long)g * st + s0 + sl);
#pragma unroll
        for (int g = 0; g < GRBW / 4; g++) vb[g] = __ldg(RB4 + (long)g * st + s0 + sl);
        const float2 csv = __ldg(reinterpret_cast<const float2 *>(W.cs) + s0 + sl);
        va[6].w = vb[GRBW / 4 - 1].z;                            // contact bits (word 12 + 3 nc + nu of the RB record)
        vb[GRBW / 4 - 1].z = csv.x; vb[GRBW / 4 - 1].w = csv.y;
#pragma unroll
        for (int g = 0; g < 7; g++) recA4[g * nsl + slot] = va[g];
#pragma unroll
        for (int g = 0; g < GRBW / 4; g++) recB4[g * nsl + slot] = vb[g];
    }
    if (C > 2) {
        const int per = (C - 2) * 144;
        const float4 *src = reinterpret_cast<const float4 *>(Psi + (long)b0 * per);
        float4 *dst = reinterpret_cast<float4 *>(psi);
        for (int i = tid; i < Gv * per / 4; i += TM_THREADS) dst[i] = __ldg(src + i);
    }
    for (int i = tid; i < Gv * (C + 1) * 12; i += TM_THREADS) {
        const int e = i / ((C + 1) * 12), r = i - e * (C + 1) * 12;
        bnd[i] = r < 12 ? x0g[(long)(b0 + e) * NX + r] : 0.0f;                          // slot 0 = x_0, slot C = 0
    }
    for (int i = tid; i < TM_CTL; i += TM_THREADS) ctl[i] = 0;
}

// ---------------------------------------------------------------------------------------------
// S3-S6: all ADMM iterations of G envs per CTA.  Warps 0-3 are the CHAIN warps (lane t of warp q = chain 32 q + t =
// TMEM lane), the others the WORKER warps: worker (slot s, quarter q, lane t) shares the TMEM lane of chain 32 q + t and
// owns stages WS s .. WS s + WS - 1 of its chunk with z, y in registers (nu = 12: three workers per chain, two stages
// each, 512 threads at 128 registers; nu = 18: two workers per chain, two stages each, 384 threads at 168 registers).
// ---------------------------------------------------------------------------------------------
template <int NU, bool WARM>
__global__ void __launch_bounds__(tm_threads(NU), 1) k_iterate_tm(SolveParams P, SrbWs W, const float *__restrict__ Psi, const float *__restrict__ x0g,
                                                              const float *__restrict__ massg, OutPtrs o, int G, int C, int has_ext,
                                                              const float *__restrict__ z0g, const float *__restrict__ y0g)
{
    constexpr int NC = NW + (NU - 12) / 3, RBW = tm_rbw(NU), GRBW = pinmpc_rb_width(NU), TM_THREADS = tm_threads(NU);
    extern __shared__ __align__(16) float smem[];
    __shared__ uint32_t tmem_slot;
    const int N = P.N, tid = threadIdx.x, lane = tid & 31;
    const int warp = tid >> 5;
    const long st = (long)P.B * N;
    const TmLay L = tm_layout(N, G, C, NU);
    const int b0 = blockIdx.x * G;
    const int Gv = min(G, P.B - b0);
    float4 *recA4 = reinterpret_cast<float4 *>(smem + L.oA), *recB4 = reinterpret_cast<float4 *>(smem + L.oB);   // [group][slot]
    float *psi = smem + L.oPsi, *bnd = smem + L.oBnd;
    const int nsl = G * N, nch = G * C, cbase = N / C, crem = N - cbase * C;      // slots, chains, stages per chunk
    // slot of stage j of chunk c of env e: stage-major over the chains; the one extra stage of the first crem chunks compacted
    auto slot_of = [&](int e, int c, int j) { return j < cbase ? j * nch + e * C + c : cbase * nch + e * crem + c; };
    int *ctl = reinterpret_cast<int *>(smem + L.oCtl);
    int *done = ctl, *ndone = ctl + 32;
    unsigned *red = reinterpret_cast<unsigned *>(ctl + 48);
    const float dt = P.dt, idt = 1.0f / P.dt;
    const int nst = Gv * N;

    // ---- tensor memory: all 512 columns (one CTA per SM) -------------------------------------------------
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"((uint32_t)__cvta_generic_to_shared(&tmem_slot)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    // ---- stage records, chunk operators, boundary slots -------------------------------------------------------
    tm_cta_load<NU>(W, Psi, x0g, st, b0, Gv, N, G, C, smem);
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tbase = tmem_slot;
    const int wq = warp & 3;
    const uint32_t myt = tbase + ((uint32_t)(wq * 32) << 16);

    // ---- the chain (env, chunk) of this TMEM lane -------------------------------------------------------------
    const int q = wq * 32 + lane;
    const int ce = q / C, cc = q - ce * C;
    const bool cvalid = ce < Gv;
    int k0 = 0, clen = 0;
    tm_chunk(N, C, cc, k0, clen);
    if (!cvalid) clen = 0;
    const int eb = cvalid ? ce : 0;
    const int sl0 = eb * N + (cvalid ? k0 : 0);                 // first stage of the chunk, CTA-local
    const int nsteps = N / C + (N % C ? 1 : 0);                  // the longest chunk
    const bool tol_mode = (P.eps_abs > 0.0f || P.eps_rel > 0.0f) && P.check_every > 0;
    if (warp < 4) {
        // =========================== CHAIN WARPS =================================================================
        tm_chain_load(W.Kh + ((long)b0 * N + sl0) * 72, has_ext ? W.c6 + ((long)b0 * N + sl0) * 6 : nullptr, clen, myt);
        tm_wait_st();
        ChainArgs A;
        A.ch.tk = myt;
        A.ch.sA = (uint32_t)__cvta_generic_to_shared(recA4 + eb * C + cc);
        A.ch.sCS = (uint32_t)__cvta_generic_to_shared(recB4 + (RBW / 4 - 1) * nsl + eb * C + cc) + 8;
        A.ch.jstride = (uint32_t)nch * 16u; A.ch.wstride = (uint32_t)nsl * 16u;
        A.ch.xoff = (uint32_t)(-(eb * (C - crem)) * 16);
        A.ch.len = clen; A.ch.nsteps = nsteps; A.ch.base = cbase;
        A.x12 = x0g[(long)(b0 + eb) * NX + 12];
        A.dt = dt; A.gdt = dt * A.x12;
        A.has_ext = has_ext; A.iters = P.iters; A.check_every = P.check_every; A.tol_mode = tol_mode; A.C = C; A.cc = cc; A.cvalid = cvalid; A.Gv = Gv;
        A.slot_lo = bnd + (eb * (C + 1) + cc) * 12;             // forward: start state; backward: own offset / true costate
        A.oxe = o.x + ((long)b0 * N + sl0) * NX;
        A.done_e = done + eb; A.ndone = ndone;
        tm_chain_main<RBW>(A);
    } else {
        // =========================== WORKER WARPS ==================================================================
        constexpr int WS = tm_lmax(NU) / tm_nwpc(NU);            // stages per worker
        const int ws = (warp - 4) >> 2;
        // Few values stay live across an iteration next to z, y of the three owned stages: everything per stage (slot,
        // contact bits, activity) is recomputed where it is used (a spilled value costs an L2 round trip here).
        const int jw = WS * ws;                                   // first owned stage of the chunk
        const int slot_x = cbase * nch + eb * crem + cc;          // slot of the chunk's extra stage (if it has one)
        const int slot_0 = eb * C + cc;                           // slot of the chunk's stage 0
        auto slot_w = [&](int a) { const int j = jw + a; return j >= clen ? slot_0 : (j < cbase ? slot_0 + j * nch : slot_x); };
        int flags = 0;                                            // bit a: stage a owned; bit 4 + a: two projections in this warp
#pragma unroll
        for (int a = 0; a < WS; a++) {
            const bool ac = jw + a < clen;
            const int bits = __float_as_int(recA4[6 * nsl + slot_w(a)].w);
            flags |= (ac ? 1 : 0) << a;
            flags |= (__any_sync(FULL, ac && (bits & 3) == 3) ? 1 : 0) << (4 + a);
        }
        const uint32_t tx = myt + TM_XOFF + 6 * jw;              // exchange vectors of the owned stages
        const uint32_t recB_u32 = (uint32_t)__cvta_generic_to_shared(recB4);
        const float m_dt = massg[b0 + eb] / dt;

        TmState<NU> S[WS];
#pragma unroll
        for (int a = 0; a < WS; a++) {
            float sv[6] = { 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f };
            const bool ac = (flags >> a) & 1;
            const long ts = (long)b0 * N + sl0 + (ac ? jw + a : 0);
#pragma unroll
            for (int j = 0; j < NU; j++) {
                S[a].z[j] = (WARM && ac) ? __ldg(z0g + ts * NU + j) : 0.0f;
                S[a].y[j] = (WARM && ac) ? __ldg(y0g + ts * NU + j) : 0.0f;
            }
            if (ac) {
                float G0[6], v[RBW];
                tm_ld_groups<0, RBW / 4>(recB_u32 + 16u * slot_w(a), 16u * nsl, v);
                tm_gh_u0<NU>(P, v + 12, S[a].z, S[a].y, G0);
                tm_sigma0<NU>(P, v, G0, idt, m_dt, sv);
            }
            tm_st6(tx + 6 * a, sv);
        }
        bool frozen = false;

        for (int it = 0; it < P.iters; it++) {
            // (uniform by construction; the modulo hides it from the compiler, the broadcast restores it)
            const bool is_check = __shfl_sync(FULL, (int)(tol_mode && ((it + 1) % P.check_every == 0)), 0) != 0;
            const bool emit = (it == P.iters - 1) || is_check;
            if (emit)
                for (int i = tid - 128; i < 5 * TM_GMAX; i += TM_THREADS - 128) red[i] = 0u;
            TM_TICK(0)
#ifdef PINMPC_TM_TIMING
            if (it == TM_TICK_IT + 1 && tid == 128) ((volatile int *)ndone)[14] = (int)clock();
#endif
            tm_sync();                                          // (1)
            __syncthreads();                                    // (2) b_c of every chunk is in the slots
            TM_TICK(1)
            // ---- backward boundary recursion: slot[c] <- Psi_c^T slot[c+1] + slot[c],  c = C-2 .. 1
            // Lane bi owns component bi.  The twelve components of the previous step are gathered from the slot itself
            // (three broadcast LDS.128 after a warp sync), column bi of Psi_c is fetched one step ahead.
            if (TM_ABL != 2 && C > 2 && lane < 24) {
                const int bsub = lane / 12, bi = lane - 12 * bsub;                       // 12 lanes per env, two envs per warp
                for (int ep = 2 * (warp - 4); ep < Gv; ep += 2 * (TM_THREADS / 32 - 4)) {                     // (an env past the end rides along)
                    const int e = ep + bsub, ee = e < Gv ? e : 0;
                    float *sb = bnd + ee * (C + 1) * 12;
                    const float *ps = psi + ee * (C - 2) * 144 + bi;
                    float m[12];
#pragma unroll
                    for (int j = 0; j < 12; j++) m[j] = ps[(C - 3) * 144 + 12 * j];
                    for (int c = C - 2; c >= 1; c--) {
                        const float4 *pv4 = reinterpret_cast<const float4 *>(sb + (c + 1) * 12);
                        const float4 p0 = pv4[0], p1 = pv4[1], p2 = pv4[2];
                        float a0 = sb[c * 12 + bi];
                        float a1 = m[1] * p0.y, a2 = m[2] * p0.z;
                        a0 = fmaf(m[0], p0.x, a0); a0 = fmaf(m[3], p0.w, a0);
                        a1 = fmaf(m[4], p1.x, a1); a2 = fmaf(m[5], p1.y, a2); a0 = fmaf(m[6], p1.z, a0); a1 = fmaf(m[7], p1.w, a1);
                        a2 = fmaf(m[8], p2.x, a2); a0 = fmaf(m[9], p2.y, a0); a1 = fmaf(m[10], p2.z, a1); a2 = fmaf(m[11], p2.w, a2);
                        if (c > 1) {
#pragma unroll
                            for (int j = 0; j < 12; j++) m[j] = ps[(c - 2) * 144 + 12 * j];
                        }
                        if (e < Gv) sb[c * 12 + bi] = a0 + (a1 + a2);
                        __syncwarp(BMASK);
                    }
                }
            }
            TM_TICK(2)
            __syncthreads();                                    // (3)
            __syncthreads();                                    // (4) d_c of every chunk is in the slots
            TM_TICK(3)
            // ---- forward boundary recursion: slot[c+1] <- Psi_c slot[c] + slot[c+1],  c = 1 .. C-2
            if (TM_ABL != 2 && C > 2 && lane < 24) {
                const int bsub = lane / 12, bi = lane - 12 * bsub;
                for (int ep = 2 * (warp - 4); ep < Gv; ep += 2 * (TM_THREADS / 32 - 4)) {
                    const int e = ep + bsub, ee = e < Gv ? e : 0;
                    float *sb = bnd + ee * (C + 1) * 12;
                    const float4 *ps = reinterpret_cast<const float4 *>(psi + ee * (C - 2) * 144 + 12 * bi);   // row bi
                    float4 m0 = ps[0], m1 = ps[1], m2 = ps[2];
                    for (int c = 1; c <= C - 2; c++) {
                        const float4 *xv4 = reinterpret_cast<const float4 *>(sb + c * 12);
                        const float4 x0 = xv4[0], x1 = xv4[1], x2 = xv4[2];
                        float a0 = sb[(c + 1) * 12 + bi];
                        float a1 = m0.y * x0.y, a2 = m0.z * x0.z;
                        a0 = fmaf(m0.x, x0.x, a0); a0 = fmaf(m0.w, x0.w, a0);
                        a1 = fmaf(m1.x, x1.x, a1); a2 = fmaf(m1.y, x1.y, a2); a0 = fmaf(m1.z, x1.z, a0); a1 = fmaf(m1.w, x1.w, a1);
                        a2 = fmaf(m2.x, x2.x, a2); a0 = fmaf(m2.y, x2.y, a0); a1 = fmaf(m2.z, x2.z, a1); a2 = fmaf(m2.w, x2.w, a2);
                        if (c < C - 2) { m0 = ps[c * 36]; m1 = ps[c * 36 + 1]; m2 = ps[c * 36 + 2]; }
                        if (e < Gv) sb[(c + 1) * 12 + bi] = a0 + (a1 + a2);
                        __syncwarp(BMASK);
                    }
                }
            }
            TM_TICK(4)
            __syncthreads();                                    // (5)
            tm_sync();                                          // (6) w of every stage is in the exchange vectors
            TM_TICK(5)
            // ---- stage update: u from w, projection, dual update, residuals, next sigma0 (one stage after the other)
            {
                float res[5] = { 0.0f, 0.0f, 0.0f, 0.0f, 0.0f };
#pragma unroll
                for (int a = 0; a < WS; a++) {
                    float wv[6];
#ifdef PINMPC_TM_UTIMING
                    int *ut = (it == TM_TICK_IT && lane == 0 && blockIdx.x == 0) ? g_ut + (warp - 4) * 32 + a * 10 : nullptr;
                    TM_UT(8)
#define TM_UTPASS , ut
#else
#define TM_UTPASS
#endif
                    tm_ld6(tx + 6 * a, wv);
                    tm_wait_ld();
                    if (((flags >> a) & 1) && TM_ABL != 1) {
                        int slot = slot_w(a);
                        asm volatile("" : "+r"(slot));             // opaque: no address of the stage record is hoisted out of the iteration loop
                        const int bits = __float_as_int(recA4[6 * nsl + slot].w);
                        const bool two = (flags >> (4 + a)) & 1;
                        if (emit) tm_stage_update<NU, true>(P, recB_u32 + 16u * slot, 16u * nsl, bits, S[a].z, S[a].y, idt, m_dt, wv, !frozen,
                                                            o.u + ((long)b0 * N + sl0 + jw + a) * NU, res, two TM_UTPASS);
                        else tm_stage_update<NU, false>(P, recB_u32 + 16u * slot, 16u * nsl, bits, S[a].z, S[a].y, idt, m_dt, wv, !frozen, nullptr, res, two TM_UTPASS);
                    } else { wv[0] = wv[1] = wv[2] = wv[3] = wv[4] = wv[5] = 0.0f; }   // unused exchange vectors stay zero
                    tm_st6(tx + 6 * a, wv);
                    asm volatile("" ::: "memory");
                    TM_UT(9)
                }
                if (emit && (flags & 1) && !frozen) {
                    atomicMax(&red[eb * 5 + 0], __float_as_uint(res[0])); atomicMax(&red[eb * 5 + 1], __float_as_uint(res[1]));
                    atomicMax(&red[eb * 5 + 2], __float_as_uint(res[2])); atomicMax(&red[eb * 5 + 3], __float_as_uint(res[3]));
                    atomicMax(&red[eb * 5 + 4], __float_as_uint(res[4]));
                }
            }
            if (emit) {
                __syncthreads();
                const int ld = tid - 128;
                if (ld < Gv && !done[ld]) {                    // one leader per env
                    const int e = ld;
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
                    frozen = done[eb] != 0;
                }
            }
        }
#pragma unroll
        for (int a = 0; a < WS; a++)
            if ((flags >> a) & 1) {
                const long ts = (long)b0 * N + sl0 + jw + a;
                constexpr int VW = NU % 4 == 0 ? 4 : 2;              // a stage's z, y start on a 48 B (nu = 12) or 72 B (nu = 18) boundary
                if (VW == 4) {
                    float4 *oz = reinterpret_cast<float4 *>(o.z + ts * NU), *oy = reinterpret_cast<float4 *>(o.y + ts * NU);
#pragma unroll
                    for (int j = 0; j < NU / 4; j++) {
                        oz[j] = make_float4(S[a].z[4 * j], S[a].z[4 * j + 1], S[a].z[4 * j + 2], S[a].z[4 * j + 3]);
                        oy[j] = make_float4(S[a].y[4 * j], S[a].y[4 * j + 1], S[a].y[4 * j + 2], S[a].y[4 * j + 3]);
                    }
                } else {
                    float2 *oz = reinterpret_cast<float2 *>(o.z + ts * NU), *oy = reinterpret_cast<float2 *>(o.y + ts * NU);
#pragma unroll
                    for (int j = 0; j < NU / 2; j++) {
                        oz[j] = make_float2(S[a].z[2 * j], S[a].z[2 * j + 1]);
                        oy[j] = make_float2(S[a].y[2 * j], S[a].y[2 * j + 1]);
                    }
                }
            }
    }
    // ---- release tensor memory ---------------------------------------------------------------------------------
    tm_sync();
#ifdef PINMPC_TM_TIMING
    if (blockIdx.x == 0 && tid == 0) {
        const int *t = ndone + 1;
        printf("chain : (1)->bwdA start %d | bwdA %d | bnd %d | bwdB %d | fwdA %d | bnd %d | fwdB %d   total %d\n", 0, t[1] - t[0], t[2] - t[1], t[3] - t[2],
               t[4] - t[3], t[5] - t[4], t[6] - t[5], t[6] - t[0]);
#ifdef PINMPC_TM_UTIMING
        for (int w = 0; w < TM_THREADS / 32 - 4; w++) {
            const int *u = g_ut + w * 32;
            printf("upd warp %2d:", w);
            for (int a = 0; a < 2; a++) {
                const int *q = u + a * 10;
                printf("  [ld %d G0 %d lam %d u %d proj %d zy %d G0n %d sig %d st %d | %d]", q[0] - q[8], q[1] - q[0], q[2] - q[1], q[3] - q[2], q[4] - q[3], q[5] - q[4],
                       q[6] - q[5], q[7] - q[6], q[9] - q[7], q[9] - q[8]);
            }
            printf("  total %d\n", u[19] - u[8]);
        }
#endif
        printf("worker: wait bwdA %d | bnd-bwd %d | wait bwdB+fwdA %d | bnd-fwd %d | wait fwdB %d | update %d   total %d\n", t[8] - t[7], t[9] - t[8],
               t[10] - t[9], t[11] - t[10], t[12] - t[11], t[13] - t[12], t[13] - t[7]);
    }
#endif
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tbase));
}

int tm_fail(pinmpc_ctx *h, const char *what, cudaError_t e)
{
    h->sticky = e;
    snprintf(h->err, sizeof h->err, "%s: %s", what, cudaGetErrorString(e));
    return -1;
}

}  // namespace

size_t pinmpc_tm_smem_bytes(int N, int G, int C, int nu) { return (size_t)tm_layout(N, G, C, nu).total * sizeof(float); }

// Chunk count and envs per CTA of the chunked kernel for this handle (0, 0 when the shape does not fit):
// C = ceil(N / 6) unless forced; G = as many envs as chains (G C <= 128), shared memory and the batch allow,
// fewest rounds of the batch over the device first, then the smallest such G (shorter boundary/update phases).
bool pinmpc_tm_config(const pinmpc_ctx *h, int *Gout, int *Cout)
{
    const int N = h->N;
    const int lmax = tm_lmax(h->nu);
    int C = h->chunks > 1 ? h->chunks : (N + lmax - 1) / lmax;
    if (C < 1 || (N + C - 1) / C > lmax || C > N || C > TM_CHAINS || C - 2 > h->psi_cap) return false;
    int best = 0;
    long best_rounds = 0;
    for (int G = 1; G <= TM_GMAX; G++) {
        if (G * C > TM_CHAINS) break;
        if (pinmpc_tm_smem_bytes(N, G, C, h->nu) + 256 > (size_t)h->smem_optin) break;
        const long per_round = (long)G * h->sm_count;
        const long rounds = (h->B + per_round - 1) / per_round;
        if (best == 0 || rounds < best_rounds) { best = G; best_rounds = rounds; }
    }
    if (h->envs_per_cta > 0 && h->envs_per_cta <= TM_GMAX && h->envs_per_cta * C <= TM_CHAINS &&
        pinmpc_tm_smem_bytes(N, h->envs_per_cta, C, h->nu) + 256 <= (size_t)h->smem_optin)
        best = h->envs_per_cta;
    if (best == 0) return false;
    *Gout = best; *Cout = C;
    return true;
}

template <int NU>
static int tm_launch_t(pinmpc_ctx *h, const SolveParams &P, const ProblemPtrs &q, int G, int C, cudaStream_t st)
{
    const int ext = q.ext != nullptr;
    auto kern = q.z0 ? k_iterate_tm<NU, true> : k_iterate_tm<NU, false>;
    const size_t smem = pinmpc_tm_smem_bytes(h->N, G, C, h->nu);
    static std::once_flag once[2];                             // process-global attribute: set once, not per solve
    static cudaError_t once_err[2];
    const int wi = q.z0 ? 1 : 0;
    std::call_once(once[wi], [&] { once_err[wi] = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, h->smem_optin - 256); });
    if (once_err[wi] != cudaSuccess) return tm_fail(h, "k_iterate_tm smem attribute", once_err[wi]);
    cudaError_t e;
    kern<<<(unsigned)((h->B + G - 1) / G), tm_threads(NU), smem, st>>>(P, h->srb, h->psi, q.x0, q.mass, h->out, G, C, ext, q.z0, q.y0);
    e = cudaGetLastError();
    if (e != cudaSuccess) return tm_fail(h, "k_iterate_tm launch", e);
    return 1;
}

// Launch the chunked iteration kernel (after assembly and factorisation, which also forms the chunk operators).
// Returns the number of kernels enqueued, or -1.
int pinmpc_launch_iterate_tm(pinmpc_ctx *h, int G, int C, cudaStream_t st)
{
    SolveParams P = make_params(h);
    ProblemPtrs q = make_problem_ptrs(h);
    return h->nu == 12 ? tm_launch_t<12>(h, P, q, G, C, st) : tm_launch_t<18>(h, P, q, G, C, st);
}
