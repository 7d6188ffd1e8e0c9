// metad_kernels.cu -- well-tempered metadynamics with the paper's two collective variables.
//   P:L136-146  V_G(s, t): Gaussians of adaptive height deposited along the CV trajectory (2 sigma in P:L140 read as 2 sigma^2)
//   P:L150-152  the CV is evaluated per bead: every bead k of a replica feels the replica's bias, F = -dV_G/ds(s_k) grad s(q_k),
//               and every deposition adds one Gaussian per bead, height (w0 / P) exp(-V_G(s_k) / (k_B T (gamma - 1)))
//   P:L164      s_dimer = d(O1,H1) - d(O2,H1) + d(O4,H2) - d(O3,H2)
//   P:L215, P:L450-452  s_water = (1/N) sum_i sum_j f_i f_j sin(Q R_ij) / (Q R_ij)  (Debye scattering intensity; all ordered pairs,
//               i = j included; minimum-image distance): an O(N^2) sum per bead with its analytic gradient
// Everything is fp64: the bias force is added to the fp64 force array after the force field.  Sums run in a fixed order.
#include "common.cuh"
#include <math.h>

namespace {

struct MdArgs {
    int N, R, P, periodic, cv, max_g;
    double box[3];
    int atoms[6];
    double f[16];
    double Q, sigma, w0, biasf, kT;
    const int *species;
    const double *q;
    double *F;
    int *n_g;
    double *gc, *gh;      // [R][max_g] centres, heights
    double *s, *dV;       // [R*P] CV value, dV_G/ds
    double *grad;         // [rows][3]
    double *partial;      // [R*P][MD_BLOCKS]
};

constexpr int MD_THREADS = 128, MD_BLOCKS_MAX = 256;

__device__ __forceinline__ double md_dist(const MdArgs &a, const double *qs, int x, int y, double u[3])
{
    double d2 = 0.0;
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) {
        double dx = qs[(size_t)x * 3 + ax] - qs[(size_t)y * 3 + ax];
        if (a.periodic) dx = dx - a.box[ax] * round(dx / a.box[ax]);
        u[ax] = dx; d2 += dx * dx;
    }
    const double d = sqrt(d2);
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) u[ax] /= d;
    return d;
}

// one thread per bead-system; the gradient array is zero outside the six atoms (cleared when the CV is enabled)
__global__ void cv_dimer_kernel(MdArgs a)
{
    const int sys = blockIdx.x * blockDim.x + threadIdx.x;
    if (sys >= a.R * a.P) return;
    const double *qs = a.q + (size_t)sys * a.N * 3;
    double *gr = a.grad + (size_t)sys * a.N * 3;
    const int pr[4][2] = {{a.atoms[0], a.atoms[1]}, {a.atoms[2], a.atoms[1]}, {a.atoms[3], a.atoms[4]}, {a.atoms[5], a.atoms[4]}};
    const double sg[4] = {1.0, -1.0, 1.0, -1.0};
    for (int k = 0; k < 6; ++k)
        for (int ax = 0; ax < 3; ++ax) gr[(size_t)a.atoms[k] * 3 + ax] = 0.0;
    double s = 0.0;
    for (int k = 0; k < 4; ++k) {
        double u[3];
        s += sg[k] * md_dist(a, qs, pr[k][0], pr[k][1], u);
        for (int ax = 0; ax < 3; ++ax) {
            gr[(size_t)pr[k][0] * 3 + ax] += sg[k] * u[ax];
            gr[(size_t)pr[k][1] * 3 + ax] -= sg[k] * u[ax];
        }
    }
    a.s[sys] = s;
}

// Debye sum: grid (blocks over atoms i, bead-system); thread = atom i walks all j through shared-memory tiles of positions
__global__ void __launch_bounds__(MD_THREADS) cv_debye_kernel(MdArgs a)
{
    __shared__ double tq[MD_THREADS][3];
    __shared__ double tf[MD_THREADS];
    __shared__ double red[MD_THREADS];
    const int sys = blockIdx.y, N = a.N;
    const double *qs = a.q + (size_t)sys * N * 3;
    const int i = blockIdx.x * MD_THREADS + threadIdx.x;
    const bool live = i < N;
    const double fi = live ? a.f[a.species[i]] : 0.0;
    double qi[3] = {0, 0, 0};
    if (live) { qi[0] = qs[(size_t)i * 3]; qi[1] = qs[(size_t)i * 3 + 1]; qi[2] = qs[(size_t)i * 3 + 2]; }
    double s = 0.0, g[3] = {0, 0, 0};
    for (int j0 = 0; j0 < N; j0 += MD_THREADS) {
        const int jl = j0 + threadIdx.x;
        __syncthreads();
        if (jl < N) { tq[threadIdx.x][0] = qs[(size_t)jl * 3]; tq[threadIdx.x][1] = qs[(size_t)jl * 3 + 1]; tq[threadIdx.x][2] = qs[(size_t)jl * 3 + 2]; tf[threadIdx.x] = a.f[a.species[jl]]; }
        __syncthreads();
        const int nj = min(MD_THREADS, N - j0);
        if (live)
            for (int t = 0; t < nj; ++t) {
                const int j = j0 + t;
                const double fj = tf[t];
                if (j == i) { s += fi * fj; continue; }
                double u[3], d2 = 0.0;
#pragma unroll
                for (int ax = 0; ax < 3; ++ax) {
                    double dx = qi[ax] - tq[t][ax];
                    if (a.periodic) dx = dx - a.box[ax] * round(dx / a.box[ax]);
                    u[ax] = dx; d2 += dx * dx;
                }
                const double R = sqrt(d2), x = a.Q * R;
                double sn, cs;
                sincos(x, &sn, &cs);
                const double sinc = sn / x;
                s += fi * fj * sinc;
                const double w = 2.0 * fi * fj * ((cs - sinc) / R) / (double)N / R;   // (2/N) f_i f_j dsinc/dR, times the unit vector u / R
#pragma unroll
                for (int ax = 0; ax < 3; ++ax) g[ax] += w * u[ax];
            }
    }
    if (live) {
        double *gr = a.grad + ((size_t)sys * N + i) * 3;
        gr[0] = g[0]; gr[1] = g[1]; gr[2] = g[2];
    }
    red[threadIdx.x] = s;
    __syncthreads();
    for (int st = MD_THREADS / 2; st > 0; st >>= 1) {
        if (threadIdx.x < st) red[threadIdx.x] += red[threadIdx.x + st];
        __syncthreads();
    }
    if (threadIdx.x == 0) a.partial[(size_t)sys * MD_BLOCKS_MAX + blockIdx.x] = red[0];
}

// per bead-system: (Debye) the block partial sums in order -> s; then V_G'(s) = -sum_g h_g (s - c_g) / sigma^2 exp(-(s - c_g)^2 / (2 sigma^2)),
// one warp per system, lanes stride over the Gaussians, fixed shuffle tree
__global__ void __launch_bounds__(32) bias_eval_kernel(MdArgs a, int n_blocks)
{
    const int sys = blockIdx.x, r = sys / a.P, lane = threadIdx.x;
    double s;
    if (a.cv == 2) {
        s = 0.0;
        for (int b = 0; b < n_blocks; ++b) s += a.partial[(size_t)sys * MD_BLOCKS_MAX + b];
        s /= (double)a.N;
        if (lane == 0) a.s[sys] = s;
    } else {
        s = a.s[sys];
    }
    const int n = a.n_g[r];
    const double is2 = 1.0 / (a.sigma * a.sigma);
    double dV = 0.0;
    for (int g = lane; g < n; g += 32) {
        const double d = s - a.gc[(size_t)r * a.max_g + g];
        dV -= a.gh[(size_t)r * a.max_g + g] * exp(-0.5 * d * d * is2) * d * is2;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dV += __shfl_xor_sync(0xffffffffu, dV, o);
    if (lane == 0) a.dV[sys] = dV;
}

__global__ void bias_force_kernel(MdArgs a)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;      // over rows * 3
    const int64_t n3 = (int64_t)a.R * a.P * a.N * 3;
    if (t >= n3) return;
    const int sys = (int)(t / ((int64_t)a.N * 3));
    a.F[t] -= a.dV[sys] * a.grad[t];
}

// one block per replica, thread = bead: height of this bead's Gaussian from the bias BEFORE the event, then append in bead order
__global__ void deposit_kernel(MdArgs a)
{
    const int r = blockIdx.x, k = threadIdx.x;
    const int n0 = a.n_g[r];
    double h = 0.0, s = 0.0;
    if (k < a.P) {
        s = a.s[(size_t)r * a.P + k];
        const double is2 = 1.0 / (a.sigma * a.sigma);
        double V = 0.0;
        for (int g = 0; g < n0; ++g) {
            const double d = s - a.gc[(size_t)r * a.max_g + g];
            V += a.gh[(size_t)r * a.max_g + g] * exp(-0.5 * d * d * is2);
        }
        h = (a.w0 / a.P) * exp(-V / (a.kT * (a.biasf - 1.0)));
    }
    __syncthreads();          // every bead has read the old Gaussians
    if (k < a.P && n0 + k < a.max_g) { a.gc[(size_t)r * a.max_g + n0 + k] = s; a.gh[(size_t)r * a.max_g + n0 + k] = h; }
    if (k == 0) a.n_g[r] = (n0 + a.P <= a.max_g) ? n0 + a.P : a.max_g;
}

MdArgs make_args(pimd_ctx *c)
{
    MdArgs a;
    const pimd_metad &m = c->md;
    a.N = c->N; a.R = c->R; a.P = c->P; a.periodic = c->periodic; a.cv = m.cv; a.max_g = PIMD_METAD_MAX;
    for (int k = 0; k < 3; ++k) a.box[k] = c->box[k];
    for (int k = 0; k < 6; ++k) a.atoms[k] = m.atoms[k];
    for (int k = 0; k < 16; ++k) a.f[k] = m.f[k];
    a.Q = m.Q; a.sigma = m.sigma; a.w0 = m.w0; a.biasf = m.biasf; a.kT = PIMD_KB * c->T;
    a.species = c->species; a.q = c->q; a.F = c->F;
    a.n_g = m.n_g; a.gc = m.gc; a.gh = m.gh; a.s = m.s; a.dV = m.dV; a.grad = m.grad; a.partial = m.partial;
    return a;
}

}  // namespace

// CV of every bead, dV_G/ds, and (add_force) F -= dV_G/ds grad s
int pimd_launch_metad_bias(pimd_ctx *c, int add_force)
{
    MdArgs a = make_args(c);
    const int nsys = c->R * c->P;
    int nb = 1;
    if (a.cv == 1) {
        cv_dimer_kernel<<<(nsys + 127) / 128, 128, 0, c->stream>>>(a);
    } else {
        nb = (c->N + MD_THREADS - 1) / MD_THREADS;
        cv_debye_kernel<<<dim3(nb, nsys), MD_THREADS, 0, c->stream>>>(a);
    }
    bias_eval_kernel<<<nsys, 32, 0, c->stream>>>(a, nb);
    c->launches += 2;
    if (add_force) {
        const int64_t n3 = c->rows * 3;
        bias_force_kernel<<<(unsigned)((n3 + 255) / 256), 256, 0, c->stream>>>(a);
        c->launches++;
    }
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}

int pimd_launch_metad_deposit(pimd_ctx *c)
{
    MdArgs a = make_args(c);
    deposit_kernel<<<c->R, ((c->P + 31) / 32) * 32, 0, c->stream>>>(a);
    c->launches++;
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}
