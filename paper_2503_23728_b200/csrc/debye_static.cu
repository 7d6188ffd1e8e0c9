// debye_static.cu -- the Debye collective variable behind an entry point that allocates nothing.
//
// pimd_debye_cv_static is for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
// loops, harnesses that forbid cudaMalloc) and have no pimd context with its caller-owned workspace at hand: same sum as
// cv_debye_kernel + bias_eval_kernel of metad_kernels.cu (same blocks of 128 atoms, same fixed order of the partial sums,
// so the same bits), but the per-block partial sums live in a file-scope device array instead of the workspace.
//   * The array is 128 KB (DEBYE_STATIC_MAX_SYS x DEBYE_STATIC_MAX_BLOCKS doubles); every GPU that loads the library holds
//     it until the process exits.  Limits: n_systems <= 256, n_atoms <= 8192 (64 blocks of 128 atoms); larger sizes are
//     rejected with PIMD_ERR_ARG.
//   * Every call shares the array and the array keeps the last call's contents.  Nothing has to start at zero: each call
//     writes every partial sum it later reads (one per (system, block)).  Calls that OVERLAP on the GPU (different streams,
//     or graph branches) race on it: serialise them.
//   * In host code `g_debye_partial` is a host-side stand-in, not a device address: the address is taken once per device,
//     with that device current, through cudaGetSymbolAddress, and passed to the kernels.
#include "common.cuh"
#include <math.h>
#include <mutex>

namespace {

constexpr int DS_THREADS = 128;
constexpr int DEBYE_STATIC_MAX_SYS = 256, DEBYE_STATIC_MAX_BLOCKS = 64, DEBYE_STATIC_MAX_SPECIES = 16;

static __device__ __align__(256) double g_debye_partial[DEBYE_STATIC_MAX_SYS * DEBYE_STATIC_MAX_BLOCKS];

struct DsArgs {
    int N, periodic;
    double box[3];
    double f[DEBYE_STATIC_MAX_SPECIES];
    double Q;
    const int *species;
    const double *q;
    double *s, *grad;       // [n_systems]; [n_systems][N][3] or null
    double *partial;        // device address of g_debye_partial
};

// grid (blocks over atoms i, bead-system); thread = atom i walks all j through shared-memory tiles of positions
__global__ void __launch_bounds__(DS_THREADS) debye_static_kernel(DsArgs a)
{
    __shared__ double tq[DS_THREADS][3];
    __shared__ double tf[DS_THREADS];
    __shared__ double red[DS_THREADS];
    const int sys = blockIdx.y, N = a.N;
    const double *qs = a.q + (size_t)sys * N * 3;
    const int i = blockIdx.x * DS_THREADS + threadIdx.x;
    const bool live = i < N;
    const double fi = live ? a.f[a.species[i]] : 0.0;
    double qi[3] = {0, 0, 0};
    if (live) { qi[0] = qs[(size_t)i * 3]; qi[1] = qs[(size_t)i * 3 + 1]; qi[2] = qs[(size_t)i * 3 + 2]; }
    double s = 0.0, g[3] = {0, 0, 0};
    for (int j0 = 0; j0 < N; j0 += DS_THREADS) {
        const int jl = j0 + threadIdx.x;
        __syncthreads();
        if (jl < N) {
            tq[threadIdx.x][0] = qs[(size_t)jl * 3]; tq[threadIdx.x][1] = qs[(size_t)jl * 3 + 1]; tq[threadIdx.x][2] = qs[(size_t)jl * 3 + 2];
            tf[threadIdx.x] = a.f[a.species[jl]];
        }
        __syncthreads();
        const int nj = min(DS_THREADS, N - j0);
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
                const double w = 2.0 * fi * fj * ((cs - sinc) / R) / (double)N / R;   // (2/N) f_i f_j dsinc/dR, times u / R
#pragma unroll
                for (int ax = 0; ax < 3; ++ax) g[ax] += w * u[ax];
            }
    }
    if (live && a.grad) {
        double *gr = a.grad + ((size_t)sys * N + i) * 3;
        gr[0] = g[0]; gr[1] = g[1]; gr[2] = g[2];
    }
    red[threadIdx.x] = s;
    __syncthreads();
    for (int st = DS_THREADS / 2; st > 0; st >>= 1) {
        if (threadIdx.x < st) red[threadIdx.x] += red[threadIdx.x + st];
        __syncthreads();
    }
    if (threadIdx.x == 0) a.partial[(size_t)sys * DEBYE_STATIC_MAX_BLOCKS + blockIdx.x] = red[0];
}

// one thread per bead-system: the block partial sums in order, divided by N
__global__ void debye_static_final_kernel(DsArgs a, int n_systems, int n_blocks)
{
    const int sys = blockIdx.x * blockDim.x + threadIdx.x;
    if (sys >= n_systems) return;
    double s = 0.0;
    for (int b = 0; b < n_blocks; ++b) s += a.partial[(size_t)sys * DEBYE_STATIC_MAX_BLOCKS + b];
    a.s[sys] = s / (double)a.N;
}

// device address of the scratch array, taken once per device with that device current
constexpr int DS_MAX_DEVICES = 64;
std::mutex g_ds_mutex;
double *g_ds_addr[DS_MAX_DEVICES] = {};

int scratch_address(double **out)
{
    int dev = -1;
    PIMD_CUDA_CHECK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= DS_MAX_DEVICES) { pimd_set_error("device ordinal %d outside [0, %d)", dev, DS_MAX_DEVICES); return PIMD_ERR_ARG; }
    std::lock_guard<std::mutex> lock(g_ds_mutex);
    if (!g_ds_addr[dev]) {
        double *p = nullptr;
        PIMD_CUDA_CHECK(cudaGetSymbolAddress((void **)&p, g_debye_partial));
        if (!p) { pimd_set_error("cudaGetSymbolAddress returned a null address for the Debye scratch array"); return PIMD_ERR_CUDA; }
        g_ds_addr[dev] = p;
    }
    *out = g_ds_addr[dev];
    return 0;
}

}  // namespace

extern "C" int pimd_debye_cv_static(const double *d_q, const int32_t *d_species, int n_atoms, int n_systems, const double box[3],
                                    const double *f_species, int n_species, double Q, double *d_s, double *d_grad, void *cuda_stream)
{
    if (!d_q || !d_species || !box || !f_species || !d_s) { pimd_set_error("null argument"); return PIMD_ERR_ARG; }
    if (n_atoms < 1 || n_systems < 1 || n_species < 1 || !(Q > 0.0)) { pimd_set_error("invalid sizes: n_atoms=%d n_systems=%d n_species=%d Q=%g", n_atoms, n_systems, n_species, Q); return PIMD_ERR_ARG; }
    const int n_blocks = (n_atoms + DS_THREADS - 1) / DS_THREADS;
    if (n_systems > DEBYE_STATIC_MAX_SYS || n_blocks > DEBYE_STATIC_MAX_BLOCKS || n_species > DEBYE_STATIC_MAX_SPECIES) {
        pimd_set_error("pimd_debye_cv_static: n_systems=%d (max %d), n_atoms=%d (max %d), n_species=%d (max %d): beyond the fixed scratch array; "
                       "use pimd_metad_cv on a context", n_systems, DEBYE_STATIC_MAX_SYS, n_atoms, DEBYE_STATIC_MAX_BLOCKS * DS_THREADS, n_species,
                       DEBYE_STATIC_MAX_SPECIES);
        return PIMD_ERR_ARG;
    }
    const bool periodic = box[0] > 0.0 && box[1] > 0.0 && box[2] > 0.0;
    if (!periodic && (box[0] != 0.0 || box[1] != 0.0 || box[2] != 0.0)) { pimd_set_error("box must be all positive or all zero"); return PIMD_ERR_ARG; }
    DsArgs a;
    a.N = n_atoms; a.periodic = periodic ? 1 : 0;
    for (int k = 0; k < 3; ++k) a.box[k] = box[k];
    for (int k = 0; k < DEBYE_STATIC_MAX_SPECIES; ++k) a.f[k] = (k < n_species) ? f_species[k] : 0.0;
    a.Q = Q; a.species = d_species; a.q = d_q; a.s = d_s; a.grad = d_grad;
    if (int rc = scratch_address(&a.partial)) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    debye_static_kernel<<<dim3(n_blocks, n_systems), DS_THREADS, 0, st>>>(a);
    debye_static_final_kernel<<<(n_systems + 127) / 128, 128, 0, st>>>(a, n_systems, n_blocks);
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}
