// nm_kernels.cu -- ring-polymer integrator kernels (rows a8-a11 of SURVEY 8(a); variants of 8(f)4).
//
// pimd_nm: one CTA owns TC (atom,dim) columns of one replica and all P beads of them, staged in
// shared memory as [P][TC] fp64 slabs; global accesses are coalesced over the column index
// (contiguous inside a bead).  The bead <-> mode maps are applied slab-wise as P x P matrices:
//   normal modes (S:N2, the default)  u = C^T q, p_u = C^T p            (orthogonal: the inverse maps are C)
//   staging                   u = F q,  p_u = F^-T p            (F from the definition of the staging variables)
//   primitive                identity; the ring springs are explicit forces in the B step
// with per-mode mass factors, frequencies and frictions set up by the host (pimd_api.cu).
// Thermostats: PILE-L (S:N3): Langevin on every mode; PILE-G: the free mode of all atoms of a replica is
// rescaled by one stochastic factor alpha (global velocity rescaling), computed by a fixed-order reduction.
// Noise is Philox4x32-10 + Box-Muller keyed by (seed; atom, r*P+mode, step, tag) (S:N4).
// HBM-bound: ~(q,p read+write, F read) 8-byte words per bead-atom-dim per step.
#include "common.cuh"
#include <math.h>

namespace {

constexpr int NM_TY = 8;

struct NmArgs {
    int N, R, P, TC;
    int transform, thermostat;   // 0 normal modes | 1 staging | 2 primitive;  0 PILE-L | 1 PILE-G
    double dt, gamma_fs, kT_P;   // kT_P = k_B T P = 1/beta_P
    double omega_P;              // P k_B T / hbar (explicit springs of the primitive variant)
    unsigned long long seed;
    const double *Tq_fwd, *Tq_inv, *Tp_fwd, *Tp_inv;   // [P][P]: u = Tq_fwd q, q = Tq_inv u, p_u = Tp_fwd p, p = Tp_inv p_u
    const double *lam, *omega_k, *gam_k;               // [P]: mode mass factor, free-ring frequency, friction (fs^-1)
    const double *mass;
    const double *alpha;         // [R] PILE-G scale of the free mode for this half-step
    double *q, *p;
    const double *F;
    int *err;
};

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// component a (0,1,2) of the three normals of counter (atom, sysmode, step, tag)  (S:N4)
__device__ __forceinline__ double normal_component(unsigned long long seed, uint32_t atom, uint32_t sysmode,
                                                   uint32_t step, uint32_t tag, int a)
{
    uint32_t x[4];
    philox4x32_10(atom, sysmode, step, tag, (uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32), x);
    const double s = 1.0 / 4294967296.0;
    const double two_pi = 6.283185307179586476925286766559;
    uint32_t xr = (a == 2) ? x[2] : x[0], xa = (a == 2) ? x[3] : x[1];
    double u1 = ((double)xr + 0.5) * s, u2 = ((double)xa + 0.5) * s;
    double rad = sqrt(-2.0 * log(u1));
    double ang = two_pi * u2;
    return rad * ((a == 1) ? sin(ang) : cos(ang));
}

// out[k][c] = sum_j M[k*P + j] * in[j][c]
__device__ __forceinline__ void xform(const double *__restrict__ M, const double *in, double *out, int P, int TC)
{
    const int c = threadIdx.x;
    // four output rows per pass: four independent accumulation chains (each in the same order j = 0 .. P-1 as a single row
    // would be, so the result is bit-identical), and one shared-memory read of in[j] serves all four
    for (int k0 = threadIdx.y; k0 < P; k0 += 4 * NM_TY) {
        const int k1 = k0 + NM_TY, k2 = k0 + 2 * NM_TY, k3 = k0 + 3 * NM_TY;
        const double *m0 = M + (size_t)k0 * P, *m1 = M + (size_t)(k1 < P ? k1 : k0) * P, *m2 = M + (size_t)(k2 < P ? k2 : k0) * P,
                     *m3 = M + (size_t)(k3 < P ? k3 : k0) * P;
        double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
        for (int j = 0; j < P; ++j) {
            const double x = in[j * TC + c];
            s0 += __ldg(m0 + j) * x;
            s1 += __ldg(m1 + j) * x;
            s2 += __ldg(m2 + j) * x;
            s3 += __ldg(m3 + j) * x;
        }
        out[k0 * TC + c] = s0;
        if (k1 < P) out[k1 * TC + c] = s1;
        if (k2 < P) out[k2 * TC + c] = s2;
        if (k3 < P) out[k3 * TC + c] = s3;
    }
}

// per-mode coefficients, formed once per CTA (they do not depend on the atom): exp(-gamma_k dt/2), sqrt(1 - that^2) for the O
// step; cos(w_k dt), sin(w_k dt) for the A step.  Same functions, same arguments as a per-thread evaluation: the same bits.
struct ModeTab { double c1[PIMD_MAX_P], c2[PIMD_MAX_P], cs[PIMD_MAX_P], sn[PIMD_MAX_P]; };

__device__ __forceinline__ void fill_mode_tab(const NmArgs &a, ModeTab &T, bool with_rotation)
{
    const double hdt = 0.5 * a.dt;
    for (int k = threadIdx.y * blockDim.x + threadIdx.x; k < a.P; k += blockDim.x * blockDim.y) {
        const double c1 = exp(-a.gam_k[k] * hdt);
        T.c1[k] = c1; T.c2[k] = sqrt(1.0 - c1 * c1);
        if (with_rotation) { double sn, cs; sincos(a.omega_k[k] * a.dt, &sn, &cs); T.cs[k] = cs; T.sn[k] = sn; }
    }
}

__device__ __forceinline__ void pile_O(const NmArgs &a, const ModeTab &T, double *pt, int r, int col, uint32_t t, uint32_t tag)
{
    const int c = threadIdx.x;
    const int atom = col / 3, dim = col - 3 * atom;
    for (int k = threadIdx.y; k < a.P; k += NM_TY) {
        if (k == 0 && a.thermostat == 1) { pt[c] = a.alpha[r] * pt[c]; continue; }   // PILE-G: one factor for the replica's free modes
        const double sig = sqrt(a.mass[atom] * a.lam[k] * a.kT_P);
        const double c1 = T.c1[k], c2 = T.c2[k];
        double xi = normal_component(a.seed, (uint32_t)atom, (uint32_t)(r * a.P + k), t, tag, dim);
        pt[k * a.TC + c] = c1 * pt[k * a.TC + c] + sig * c2 * xi;
    }
}

// B(dt/2) of the primitive variant adds the explicit ring springs -m w_P^2 ((q_j - q_{j-1}) + (q_j - q_{j+1}))
__device__ __forceinline__ double spring_force(const NmArgs &a, const double *bQ, int j, int c, double mi)
{
    const int P = a.P, jm = (j + P - 1) % P, jp = (j + 1) % P;
    const double qj = bQ[j * a.TC + c];
    return -mi * a.omega_P * a.omega_P * ((qj - bQ[jm * a.TC + c]) + (qj - bQ[jp * a.TC + c]));
}

// mode: 0 = pre (O,B,A), 1 = post (B,O), 2 = initial momenta (S:N5)
// The step index of the noise counter is read from device memory (t = *t_dev - t_off; null = 0), so that the launch sequence
// of one step does not depend on the step and can be captured once as a CUDA graph and replayed.
__device__ __forceinline__ uint32_t step_of(const uint32_t *t_dev, uint32_t t_off) { return t_dev ? *t_dev - t_off : 0u; }

__global__ void step_set_kernel(uint32_t *t_dev, uint32_t t) { pdl_enter(); t_dev[0] = t; t_dev[1] = t; }

template <int MODE>
__global__ void __launch_bounds__(32 * NM_TY) nm_kernel(NmArgs a, const uint32_t *t_dev, uint32_t t_off, uint32_t *t_next)
{ pdl_enter();
    const uint32_t t = step_of(t_dev, t_off);
    // The step counter lives in two device words that the two halves of a step hand to each other: the first half reads word 0 and
    // leaves t + 1 in word 1, the second half reads word 1 (minus one) and leaves t + 1 in word 0.  Nothing reads the word a kernel
    // writes while that kernel runs, and no separate increment kernel is needed.
    if (t_next && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0 && threadIdx.y == 0) *t_next = t + 1u;
    extern __shared__ double sm[];
    const int P = a.P, TC = a.TC;
    double *bP = sm, *bT = sm + (size_t)P * TC, *bQ = bT + (size_t)P * TC, *bQ2 = bQ + (size_t)P * TC;
    const int c = threadIdx.x, r = blockIdx.y;
    const int ncol = 3 * a.N;
    const int col = blockIdx.x * TC + c;
    const bool live = col < ncol;
    const int colc = live ? col : 0;
    const size_t base = (size_t)r * P * ncol + colc;
    const bool thermo = a.gamma_fs >= 0.0;
    const double hdt = 0.5 * a.dt;

    if (MODE == 2) {
        const int atom = colc / 3, dim = colc - 3 * atom;
        for (int k = threadIdx.y; k < P; k += NM_TY)
            bT[k * TC + c] = sqrt(a.mass[atom] * a.lam[k] * a.kT_P) * normal_component(a.seed, (uint32_t)atom, (uint32_t)(r * P + k), 0u, 2u, dim);
        __syncthreads();
        xform(a.Tp_inv, bT, bP, P, TC);
        __syncthreads();
        if (live)
            for (int j = threadIdx.y; j < P; j += NM_TY) a.p[base + (size_t)j * ncol] = bP[j * TC + c];
        return;
    }

    __shared__ ModeTab tab;
    fill_mode_tab(a, tab, MODE == 0);              // (read after at least one __syncthreads below)
    bool bad = false;
    const bool prim = a.transform == 2;
    const double mi = a.mass[colc / 3];
    if (MODE == 0 || prim) {
        for (int j = threadIdx.y; j < P; j += NM_TY) bQ[j * TC + c] = live ? a.q[base + (size_t)j * ncol] : 0.0;
        if (MODE == 1) __syncthreads();   // the spring force below reads the neighbouring beads
    }
    for (int j = threadIdx.y; j < P; j += NM_TY) {
        double pv = live ? a.p[base + (size_t)j * ncol] : 0.0;
        if (MODE == 1) {  // B(dt/2) first
            double f = live ? a.F[base + (size_t)j * ncol] : 0.0;
            bad |= !isfinite(f);
            if (prim) f += spring_force(a, bQ, j, c, mi);
            pv += hdt * f;
        }
        bP[j * TC + c] = pv;
    }
    __syncthreads();
    if (thermo) {
        xform(a.Tp_fwd, bP, bT, P, TC);
        __syncthreads();
        pile_O(a, tab, bT, r, colc, t, MODE == 0 ? 0u : 1u);
        __syncthreads();
        xform(a.Tp_inv, bT, bP, P, TC);
        __syncthreads();
    }
    if (MODE == 1) {
        if (live)
            for (int j = threadIdx.y; j < P; j += NM_TY) a.p[base + (size_t)j * ncol] = bP[j * TC + c];
        if (bad) atomicOr(a.err, PIMD_FLAG_NAN);
        return;
    }
    // MODE 0: B(dt/2), then A(dt): every mode is propagated exactly under p^2 / (2 m lam) + 1/2 m lam w^2 u^2
    for (int j = threadIdx.y; j < P; j += NM_TY) {
        double f = live ? a.F[base + (size_t)j * ncol] : 0.0;
        if (prim) f += spring_force(a, bQ, j, c, mi);
        bP[j * TC + c] += hdt * f;
    }
    __syncthreads();
    xform(a.Tq_fwd, bQ, bQ2, P, TC);
    xform(a.Tp_fwd, bP, bT, P, TC);
    __syncthreads();
    {
        for (int k = threadIdx.y; k < P; k += NM_TY) {
            double qt = bQ2[k * TC + c], pt = bT[k * TC + c];
            const double mu = mi * a.lam[k], w = a.omega_k[k];
            if (w == 0.0) {
                qt = qt + a.dt * pt / mu;
            } else {
                const double sn = tab.sn[k], cs = tab.cs[k];
                double pn = cs * pt - mu * w * sn * qt;
                double qn = sn / (mu * w) * pt + cs * qt;
                pt = pn; qt = qn;
            }
            bQ2[k * TC + c] = qt; bT[k * TC + c] = pt;
        }
    }
    __syncthreads();
    xform(a.Tq_inv, bQ2, bQ, P, TC);
    xform(a.Tp_inv, bT, bP, P, TC);
    __syncthreads();
    if (live)
        for (int j = threadIdx.y; j < P; j += NM_TY) {
            double qv = bQ[j * TC + c];
            bad |= !isfinite(qv);
            a.q[base + (size_t)j * ncol] = qv;
            a.p[base + (size_t)j * ncol] = bP[j * TC + c];
        }
    if (bad) atomicOr(a.err, PIMD_FLAG_NAN);
}

// PILE-G (global thermostat on the free modes of a replica): per replica, the kinetic energy K of the free
// modes (k = 0) of all atoms, and the noise sums R1 (first normal: atom 0, x) and S (squares of the other 3N - 1 normals of
// the stream PILE-L would use for mode 0).  Partial sums per block in a fixed order, then one thread per replica:
//   alpha^2 = c + (1 - c) (R1^2 + S) / (2 beta_P K) + 2 R1 sqrt(c (1 - c) / (2 beta_P K)),  c = exp(-gamma dt / 2),
//   sign(alpha) = sign(R1 + sqrt(2 beta_P K c / (1 - c)))           (stochastic velocity rescaling, exact for the half-step)
constexpr int PG_BLOCKS = 64, PG_THREADS = 128;

__global__ void __launch_bounds__(PG_THREADS) pileg_partial_kernel(NmArgs a, const uint32_t *t_dev, uint32_t t_off, uint32_t tag, int after_B, double *__restrict__ partial)
{ pdl_enter();
    const uint32_t t = step_of(t_dev, t_off);
    __shared__ double red[2][PG_THREADS];
    const int r = blockIdx.y, P = a.P, ncol = 3 * a.N;
    const double hdt = 0.5 * a.dt;
    double K = 0.0, S = 0.0;
    for (int col = blockIdx.x * PG_THREADS + threadIdx.x; col < ncol; col += PG_BLOCKS * PG_THREADS) {
        const int atom = col / 3, dim = col - 3 * atom;
        const size_t base = (size_t)r * P * ncol + col;
        double pm = 0.0;
        for (int j = 0; j < P; ++j) {
            double pv = a.p[base + (size_t)j * ncol];
            if (after_B) pv += hdt * a.F[base + (size_t)j * ncol];
            pm += a.Tp_fwd[j] * pv;          // row 0 of the momentum map: the free mode
        }
        K += pm * pm / (2.0 * a.mass[atom] * a.lam[0]);
        if (col > 0) {
            const double xi = normal_component(a.seed, (uint32_t)atom, (uint32_t)(r * P), t, tag, dim);
            S += xi * xi;
        }
    }
    red[0][threadIdx.x] = K; red[1][threadIdx.x] = S;
    __syncthreads();
    for (int s = PG_THREADS / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) { red[0][threadIdx.x] += red[0][threadIdx.x + s]; red[1][threadIdx.x] += red[1][threadIdx.x + s]; }
        __syncthreads();
    }
    if (threadIdx.x < 2) partial[((size_t)r * PG_BLOCKS + blockIdx.x) * 2 + threadIdx.x] = red[threadIdx.x][0];
}

__global__ void pileg_final_kernel(NmArgs a, const uint32_t *t_dev, uint32_t t_off, uint32_t tag, const double *__restrict__ partial, double *__restrict__ alpha)
{ pdl_enter();
    const uint32_t t = step_of(t_dev, t_off);
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= a.R) return;
    double K = 0.0, S = 0.0;
    for (int b = 0; b < PG_BLOCKS; ++b) { K += partial[((size_t)r * PG_BLOCKS + b) * 2]; S += partial[((size_t)r * PG_BLOCKS + b) * 2 + 1]; }
    const double R1 = normal_component(a.seed, 0u, (uint32_t)(r * a.P), t, tag, 0);
    const double c1 = exp(-a.gamma_fs * 0.5 * a.dt), bP = 1.0 / a.kT_P;
    double al = 1.0;
    if (K > 0.0) {
        const double a2 = c1 + (1.0 - c1) * (R1 * R1 + S) / (2.0 * bP * K) + 2.0 * R1 * sqrt(c1 * (1.0 - c1) / (2.0 * bP * K));
        const double sgn = (R1 + sqrt(2.0 * bP * K * c1 / (1.0 - c1)) >= 0.0) ? 1.0 : -1.0;
        al = sgn * sqrt(a2 > 0.0 ? a2 : 0.0);
    }
    alpha[r] = al;
}

NmArgs make_args(const pimd_ctx *c)
{
    NmArgs a;
    a.N = c->N; a.R = c->R; a.P = c->P; a.TC = (c->P <= 128) ? 32 : 16;
    a.transform = c->transform; a.thermostat = c->thermostat;
    a.dt = c->dt; a.gamma_fs = c->gamma_fs; a.kT_P = PIMD_KB * c->T * c->P;
    a.omega_P = c->P * PIMD_KB * c->T / PIMD_HBAR;
    a.seed = c->seed;
    a.Tq_fwd = c->Tq_fwd; a.Tq_inv = c->Tq_inv; a.Tp_fwd = c->Tp_fwd; a.Tp_inv = c->Tp_inv;
    a.lam = c->lam_k; a.omega_k = c->omega_k; a.gam_k = c->gam_k; a.mass = c->mass; a.alpha = c->pileg_alpha;
    a.q = c->q; a.p = c->p; a.F = c->F; a.err = c->err;
    return a;
}

template <int MODE>
int launch_nm(pimd_ctx *c, const uint32_t *t_dev, uint32_t t_off, uint32_t *t_next)
{
    NmArgs a = make_args(c);
    if (MODE != 2 && c->thermostat == 1 && c->gamma_fs >= 0.0) {   // PILE-G: the replica's scale factor for this half-step
        const uint32_t tag = MODE == 0 ? 0u : 1u;
        pimd_launch(pileg_partial_kernel, dim3(PG_BLOCKS, c->R), PG_THREADS, 0, c->stream, a, t_dev, t_off, tag, MODE == 1 ? 1 : 0, c->pileg_partial);
        pimd_launch(pileg_final_kernel, (c->R + 127) / 128, 128, 0, c->stream, a, t_dev, t_off, tag, c->pileg_partial, c->pileg_alpha);
        c->launches += 2;
    }
    size_t smem = (size_t)4 * c->P * a.TC * sizeof(double);
    if (!(c->attr_done & ATTR_NM)) {   // all three variants at once (no attribute call inside a stream capture)
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(nm_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(nm_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(nm_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        c->attr_done |= ATTR_NM;
    }
    dim3 grid((3 * c->N + a.TC - 1) / a.TC, c->R), block(a.TC, NM_TY);
    pimd_launch(nm_kernel<MODE>, grid, block, smem, c->stream, a, t_dev, t_off, t_next);
    c->launches++;
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}

// ---------------------------------------------------------------------------------------------
__global__ void simple_forces_kernel(int kind, int N, int64_t n3, double w2, const double *__restrict__ mass,
                                     const double *__restrict__ q, double *__restrict__ F)
{ pdl_enter();
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n3) return;
    if (kind == 2) { F[t] = 0.0; return; }
    int atom = (int)((t / 3) % N);
    F[t] = -(mass[atom] * w2) * q[t];
}

__global__ void copy_forces_f32_kernel(int64_t n3, const double *__restrict__ F, float *__restrict__ out)
{
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n3) out[t] = (float)F[t];
}

// estimators (S:E1-E4): partial sums per (replica, block of atoms), fixed-order tree reduction
constexpr int EST_BLOCKS = 64, EST_THREADS = 128;

__global__ void __launch_bounds__(EST_THREADS)
estimators_partial_kernel(int N, int P, int kind, double omega_P, double w_h, const double *__restrict__ mass,
                          const double *__restrict__ q, const double *__restrict__ p, const double *__restrict__ F,
                          double *__restrict__ partial)
{
    __shared__ double red[5][EST_THREADS];
    const int r = blockIdx.y;
    double acc[5] = {0, 0, 0, 0, 0};  // spring, vir, cvir, vpot, tc
    for (int i = blockIdx.x * EST_THREADS + threadIdx.x; i < N; i += EST_BLOCKS * EST_THREADS) {
        const double mi = mass[i];
        double qbar[3] = {0, 0, 0}, pc[3] = {0, 0, 0};
        for (int k = 0; k < P; ++k) {
            size_t o = (((size_t)r * P + k) * N + i) * 3;
            for (int a = 0; a < 3; ++a) { qbar[a] += q[o + a]; pc[a] += p[o + a]; }
        }
        const double rs = 1.0 / sqrt((double)P);
        for (int a = 0; a < 3; ++a) { qbar[a] /= P; pc[a] *= rs; }
        for (int k = 0; k < P; ++k) {
            size_t o = (((size_t)r * P + k) * N + i) * 3;
            size_t on = (((size_t)r * P + (k + 1) % P) * N + i) * 3;
            for (int a = 0; a < 3; ++a) {
                double qk = q[o + a], dq = qk - q[on + a], f = F[o + a];
                acc[0] += 0.5 * mi * omega_P * omega_P * dq * dq;
                acc[1] += qk * f;
                acc[2] += (qk - qbar[a]) * f;
                if (kind == 1) acc[3] += 0.5 * mi * w_h * w_h * qk * qk;
            }
        }
        for (int a = 0; a < 3; ++a) acc[4] += pc[a] * pc[a] / mi;
    }
    for (int v = 0; v < 5; ++v) red[v][threadIdx.x] = acc[v];
    __syncthreads();
    for (int s = EST_THREADS / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s)
            for (int v = 0; v < 5; ++v) red[v][threadIdx.x] += red[v][threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x < 5) partial[((size_t)r * EST_BLOCKS + blockIdx.x) * 8 + threadIdx.x] = red[threadIdx.x][0];
}

__global__ void estimators_final_kernel(int R, int N, int P, int kind, double kT, const double *__restrict__ partial,
                                        double *__restrict__ out)
{
    int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    double s[5] = {0, 0, 0, 0, 0};
    for (int b = 0; b < EST_BLOCKS; ++b)
        for (int v = 0; v < 5; ++v) s[v] += partial[((size_t)r * EST_BLOCKS + b) * 8 + v];
    out[r * 8 + 0] = 1.5 * N * P * kT - s[0] / P;
    out[r * 8 + 1] = -s[1] / (2.0 * P);
    out[r * 8 + 2] = 1.5 * N * kT - s[2] / (2.0 * P);
    out[r * 8 + 3] = (kind == 0) ? nan("") : s[3] / P;
    out[r * 8 + 4] = s[4] / (3.0 * N * PIMD_KB * P);
}

}  // namespace

int pimd_launch_init_momenta(pimd_ctx *c) { return launch_nm<2>(c, nullptr, 0u, nullptr); }
// device step counter: word 0 holds t at the start of a step, word 1 holds t + 1 between the two halves (see nm_kernel)
int pimd_launch_nm_pre(pimd_ctx *c) { return launch_nm<0>(c, c->step_dev, 0u, c->step_dev + 1); }
int pimd_launch_nm_post(pimd_ctx *c) { return launch_nm<1>(c, c->step_dev + 1, 1u, c->step_dev); }
int pimd_launch_set_step(pimd_ctx *c, uint32_t t)
{
    pimd_launch(step_set_kernel, 1, 1, 0, c->stream, c->step_dev, t);
    c->launches++;
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}

int pimd_launch_simple_forces(pimd_ctx *c)
{
    int64_t n3 = c->rows * 3;
    double w2 = c->harmonic_omega * c->harmonic_omega;
    pimd_launch(simple_forces_kernel, (unsigned)((n3 + 255) / 256), 256, 0, c->stream, c->kind, c->N, n3, w2, c->mass, c->q, c->F);
    c->launches++;
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}

int pimd_launch_copy_forces_f32(pimd_ctx *c, float *d_out)
{
    int64_t n3 = c->rows * 3;
    copy_forces_f32_kernel<<<(unsigned)((n3 + 255) / 256), 256, 0, c->stream>>>(n3, c->F, d_out);
    c->launches++;
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}

int pimd_launch_estimators(pimd_ctx *c)
{
    double kT = PIMD_KB * c->T, omega_P = c->P * kT / PIMD_HBAR;
    estimators_partial_kernel<<<dim3(EST_BLOCKS, c->R), EST_THREADS, 0, c->stream>>>(
        c->N, c->P, c->kind, omega_P, c->harmonic_omega, c->mass, c->q, c->p, c->F, c->est_partial);
    estimators_final_kernel<<<(c->R + 127) / 128, 128, 0, c->stream>>>(c->R, c->N, c->P, c->kind, kT, c->est_partial,
                                                                        c->est_out);
    c->launches += 2;
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}
