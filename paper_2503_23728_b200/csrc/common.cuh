// common.cuh -- shared declarations of the sm_100a PIMD library (host context, device views).
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda.h>            // CUtensorMap (type only: the encoder is fetched through cudaGetDriverEntryPoint)
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/pimd.h"

// CODATA 2018; hard-coded independently of the oracle.
#define PIMD_KB 8.617333262145e-5      // eV / K
#define PIMD_HBAR 0.658211956548       // eV fs
#define PIMD_AMU 103.6426965268        // 1 amu A^2/fs^2 in eV

#define PIMD_MAX_P 256
#define PIMD_MAX_NBR 512               // neighbours per atom the fill kernel can sort

// device error word bits
#define PIMD_FLAG_PAIRS 1
#define PIMD_FLAG_NAN 2

struct GfnLayerW {
    const float *WsT, *WvnT, *WvmT, *bv1, *Wv2T, *bv2, *WaT, *ba;  // transposed [in][out]
};

// Device-side view of the network (all pointers into the workspace).
struct GfnDev {
    int S, K, H, L;
    float r_cut, agg_norm, force_scale;
    const float *Emb;                  // [S][H]
    const float *We1T, *be1;           // [K][H]
    const float *We2T, *be2;           // [H][H]
    const float *WfeT, *bfe;           // (W_f1 W_e2)^T [H][H], W_f1 b_e2 + b_f1
    const float *Wf1T;                 // [H][H]  (G = W_f1 E)
    const float *wf2;                  // [H]
    float bf2;
    GfnLayerW layer[8];
};

struct NlistDev {
    int ncell[3];
    int ncell_tot;                     // per bead-system
    int *cell_id;                      // [rows]
    int *cell_count;                   // [nsys*ncell_tot]
    int *cell_start;                   // [nsys*(ncell_tot+1)] relative to the system's first row
    int *cell_cursor;                  // [nsys*ncell_tot]
    int *sorted_atom;                  // [rows] local atom index in cell order
    double *sorted_q;                  // [rows][3]
    int *nnz;                          // [rows] neighbours within r_cut (this step)
    int *ncand;                        // [rows] candidates within r_cut + skin (since the last rebuild)
    int *hits;                         // [rows][hit_stride] candidate indices of each row, ascending j after the rebuild
    unsigned *hitmask;                 // [rows][PIMD_MAX_NBR / 32] which candidates are within r_cut this step
    double *q_ref;                     // [rows][3] positions the candidate lists were built at
    float4 *q32;                       // [rows] fp32 copy of the current positions (filter estimate)
    int *need;                         // device flag: rebuild the candidate lists
    double skin;                       // A; 0 = rebuild every step
    int hit_stride;
    int *row_ptr;                      // [rows+1]
    int *block_sums;                   // [ceil(rows/1024)+1]
    int *col;                          // [pair_cap] local atom index j
    int *pair_row;                     // [pair_cap] global row i
    float4 *dvec;                      // tcgen05 pipeline only, else null: [pair_cap] r_j - r_i (fp64 difference, minimum image,
                                       // then fp32) | segment kind of the row inside the pair's 32-pair granule (int bits)
    int64_t pair_cap;
};

#define PIMD_METAD_MAX 16384           // Gaussians per replica the workspace holds
#define PIMD_METAD_BLOCKS 256          // partial sums per bead-system of the Debye CV (N <= 32768)

// well-tempered metadynamics: one bias per replica, felt by every bead
struct pimd_metad {
    int cv;                            // 0 off, 1 s_dimer, 2 Debye
    int atoms[6];
    double f[16], Q, sigma, w0, biasf;
    int every;
    int *n_g;                          // [R]
    double *gc, *gh;                   // [R][PIMD_METAD_MAX]
    double *s, *dV;                    // [R*P]
    double *grad;                      // [rows][3]
    double *partial;                   // [R*P][PIMD_METAD_BLOCKS]
};

struct pimd_ctx {
    int N, R, P, periodic;
    int64_t rows;                      // R*P*N
    double box[3];
    double T, dt, gamma_fs;            // gamma_fs < 0: NVE
    uint64_t seed;
    int64_t step;
    int kind, gemm_dtype, n_species_host;
    double harmonic_omega;
    cudaStream_t stream;
    int forces_valid;
    int64_t launches, launches_per_step;
    int num_sms;
    int device;                        // CUDA device the workspace and stream belong to (set current at every entry point)
    unsigned attr_done;                // per-context (= per-device) bits: opt-in shared-memory attribute set for a kernel family

    // workspace views
    double *q, *p, *F;                 // [rows][3]
    int *species;                      // [N]
    double *mass;                      // [N] internal units
    int transform, thermostat;         // integrator variant (pimd_set_integrator): 0 normal modes | 1 staging | 2 primitive; 0 PILE-L | 1 PILE-G
    double *Cmat, *CmatT;              // [P][P]: C[j*P+k]; CT[k*P+j]   (normal-mode matrix, S:N2)
    double *Tq_fwd, *Tq_inv, *Tp_fwd, *Tp_inv;   // [P][P] bead <-> mode maps of coordinates and momenta in use
    double *Tstage;                    // [4][P][P] the staging maps (used when transform == 1)
    double *omega_k, *lam_k, *gam_k;   // [P] mode frequency, mass factor, friction
    double *pileg_partial, *pileg_alpha;   // [R][64][2], [R]
    int *err;                          // [4] device error word
    uint32_t *step_dev;                // two device words of the step counter (read by the noise kernels: a captured step does not depend on it)
    cudaGraphExec_t step_graph;        // one whole step, captured at the first pimd_step (null: not captured yet)
    int graph_state;                   // 0 not tried, 1 captured, -1 capture not available
    int warm;                          // a step has run with plain launches (every lazy kernel attribute is set)
    double *est_partial;               // [R][EST_BLOCKS][8]
    double *est_out;                   // [R][8]
    NlistDev nl;
    GfnDev net;
    float *weights_dev;                // raw + derived weights
    uint16_t *wimg_wf2;                // bf16 UMMA image of w_f2 replicated on 16 rows (readout product of the head)
    uint16_t *wimg_e1, *wimg_e2, *wimg_fe;   // bf16 UMMA images (K-major, 128B swizzle) for the tcgen05 path
    int use_tc;                        // 1: tensor-core pair and node kernels (gemm_dtype 1, K=64, H=128)
    uint16_t *wimg_node;               // [L][20] bf16 UMMA half-images (16 KB): (W_vn/2, W_vm/2, W_v2, W_a, W_s^{l+1} or W_f1) x (hi, lo) x 2 K blocks
    float *xs0;                        // [S][H] W_s^0 Emb[s]
    float h_be1_half[128];             // HOST copy of b_e1 / 2 (passed to the pair kernels as kernel parameters)
    unsigned char *h1_img, *meta_img;  // [pair_cap/128 + 1] tile images kept between the pair passes of one evaluation (tc path)
    bool nl_flag_up = false;           // host mirror: the rebuild flag of the neighbour list is known to be raised (direct path: it stays so)
    uint32_t *XE;                      // [rows][H] words gathered by the pair kernels: x bf16 in the low half, the word as fp32 = E x (tc::pack_x_y); aliases xfeat
    CUtensorMap tmap_xe, tmap_g;       // 2-D tensor maps [rows][128 x 32 bit] of XE and G for TMA tile::gather4 (four gathered rows per copy)
    float *nfeat, *xfeat, *mfeat, *Efeat, *Gfeat;   // [rows][H]
    float *carry_m;                    // [n_gran_m][2][H]
    float *carry_f;                    // [n_gran_f][2][4]
    float *Fraw;                       // [rows][4] complete-row partial force sums
    int gran_m, gran_f;                // pairs per reduction granule
    int64_t n_gran_m, n_gran_f;
    pimd_metad md;
    struct PimdProf *prof;             // host-side event recorder (pimd_profile)
};

// records a CUDA event pair on the context's stream around the launches made in its scope
void pimd_prof_begin(pimd_ctx *c, int kind);
void pimd_prof_end(pimd_ctx *c);
struct ProfScope {
    pimd_ctx *c;
    ProfScope(pimd_ctx *ctx, int kind) : c(ctx) { if (c->prof) pimd_prof_begin(c, kind); }
    ~ProfScope() { if (c->prof) pimd_prof_end(c); }
};
enum { ATTR_PAIR32 = 1, ATTR_NODE32 = 2, ATTR_PIPE = 4, ATTR_NODETC = 8, ATTR_FILL = 16, ATTR_SORT = 32, ATTR_NM = 256 /* << MODE */ };
enum { PROF_NM = 0, PROF_NLIST = 1, PROF_PAIR = 2, PROF_NODE = 3, PROF_HEAD = 4, PROF_OTHER = 5 };

void pimd_set_error(const char *fmt, ...);

#define PIMD_CUDA_CHECK(call)                                                            \
    do {                                                                                 \
        cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess) {                                                         \
            pimd_set_error("%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            return PIMD_ERR_CUDA;                                                        \
        }                                                                                \
    } while (0)

// Programmatic dependent launch: every kernel of the step is launched with programmatic stream serialisation, so that its
// launch is processed while the kernel before it still runs and it starts the moment that one ends -- in a captured graph too
// (ice512 -2 %, fad_p8 -17 % per step).  A kernel so launched must not touch memory written by its predecessors before
// pdl_enter() (griddepcontrol.wait returns when the grids before it have completed and flushed): it is the first statement of
// every such kernel.  No kernel triggers its dependents early (griddepcontrol.launch_dependents): measured, early-resident
// blocks of the next kernel cost fad_x64_p32 +26 % per step and ice512 gained nothing over the implicit trigger at exit.
// Nor does it pay in the two big persistent kernels alone (trigger at entry, wait after barrier initialisation, TMEM allocation and
// the copies of the static weights, so that the next kernel's blocks set themselves up on SMs whose block has finished): ice512 +4 %.
#if defined(__CUDACC__)
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_enter() { pdl_wait(); }

template <typename... KArgs, typename... Args>
static inline cudaError_t pimd_launch(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}
#endif

// kernel launchers (each returns 0 or PIMD_ERR_CUDA)
int pimd_launch_init_momenta(pimd_ctx *c);
int pimd_launch_nm_pre(pimd_ctx *c);                 // O B A with the noise of step step_dev[0]; leaves step_dev[1] = that + 1
int pimd_launch_set_step(pimd_ctx *c, uint32_t t);   // step_dev[0] = step_dev[1] = t
int pimd_launch_nm_post(pimd_ctx *c);                // B O with the noise of step step_dev[1] - 1; leaves step_dev[0] = step_dev[1]
int pimd_launch_simple_forces(pimd_ctx *c);          // kinds 1, 2
int pimd_launch_estimators(pimd_ctx *c);
int pimd_launch_nlist(pimd_ctx *c);
int pimd_launch_nlist_invalidate(pimd_ctx *c);       // positions were replaced from outside: rebuild the candidate lists
int pimd_launch_gfn_forces(pimd_ctx *c);
int pimd_launch_metad_bias(pimd_ctx *c, int add_force);   // CV and dV_G/ds of every bead; add_force: F -= dV_G/ds grad s
int pimd_launch_metad_deposit(pimd_ctx *c);               // one Gaussian per bead at the CV values of the last evaluation
int pimd_launch_copy_forces_f32(pimd_ctx *c, float *d_out);
size_t pimd_gfn_smem_bytes(int K, int H);
bool pimd_gfn_supported(int K, int H);

static inline size_t pimd_align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }
