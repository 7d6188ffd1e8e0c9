/*
 * pimd.h -- C-ABI of the B200-native PIMD hot path (libpimd_b200.so).
 *
 * One ring-polymer path-integral MD step over all P beads, as stated in
 * arXiv 2503.23728 (citations "P:Lnnn" = line of the paper text, "S:x" = reading
 * listed in DESIGN.md / SURVEY.md section 8(c)):
 *
 *   (a) per-bead periodic cell-list neighbour build        (cutoff only: P:L394)
 *   (b) bead-batched, back-propagation-free GFN force net   (eqs; S:G0-G6)
 *   (c) normal-mode transform, exact free-ring-polymer step
 *       and PILE-L thermostat with Philox noise            (S:N1-N5)
 *
 * Every step runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.
 * No torch / C++ types cross this boundary: plain pointers and sizes only.  Each
 * pointer argument says whether it is HOST or DEVICE memory.
 *
 * Units: Angstrom, fs, amu, K, eV, eV/A; centroid friction in ps^-1.
 * Layout: every per-bead array is [replica][bead][atom][xyz], row id = (r*P + k)*N + i.
 *
 * Errors: every call returns 0 on success or
 *   PIMD_ERR_ARG   (-1) invalid argument (null pointer, P < 1 or > 256, periodic box edge
 *                        < 2 r_cut, weight count mismatch, workspace too small, unsupported
 *                        (n_rbf, hidden) pair)
 *   PIMD_ERR_CUDA  (-2) a CUDA call failed
 *   PIMD_ERR_PAIRS (-3) pair capacity (or 512 neighbours per atom) exceeded
 *   PIMD_ERR_NAN   (-4) non-finite force or position met on the device
 * Device-detected conditions (-3, -4) are latched in a device word and returned by the
 * next synchronising call (pimd_estimators, pimd_get_state, pimd_nlist, pimd_sync).
 * pimd_last_error() returns a thread-local description.  After an error the context is
 * only good for pimd_destroy.
 */
#ifndef PIMD_B200_H
#define PIMD_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PIMD_OK 0
#define PIMD_ERR_ARG (-1)
#define PIMD_ERR_CUDA (-2)
#define PIMD_ERR_PAIRS (-3)
#define PIMD_ERR_NAN (-4)

typedef struct pimd_ctx pimd_ctx; /* opaque; host object that owns nothing but views into the workspace */

/* Network / potential description.  `weights` is a HOST pointer, copied by pimd_create. */
typedef struct {
    int32_t kind;       /* 0 GFN net; 1 harmonic test well V = 1/2 m w^2 |r|^2 per atom;
                           2 none (free ring polymer) */
    int32_t n_species;  /* S */
    int32_t n_rbf;      /* K  Gaussian radial basis functions on [0, r_cut] (S:G1) */
    int32_t hidden;     /* H  feature width ("Feat. Dim.") */
    int32_t n_layers;   /* L  interaction layers ("N_inter") */
    int32_t gemm_dtype; /* 0: fp32 everywhere.  1: bf16 operands + fp32 accumulation on the
                           tensor cores for the dense contractions (tolerance 2e-2) */
    float r_cut;        /* A (0.6 nm) */
    float agg_norm;     /* constant multiplying every neighbour sum (S:G6) */
    float force_scale;  /* eV/A per unit network output (S:G6) */
    double harmonic_omega; /* rad/fs, kind 1 only */
    const float *weights;  /* HOST, packed fp32 in the order of S:G0:
                              Emb[S][H]; W_e1[H][K], b_e1[H], W_e2[H][H], b_e2[H];
                              per layer: W_s, W_vn, W_vm [H][H], b_v1[H], W_v2[H][H], b_v2[H], W_a[H][H], b_a[H];
                              W_f1[H][H], b_f1[H], w_f2[H], b_f2[1]; matrices row-major [out][in] */
    int64_t n_weights;
} pimd_net_params;

/* Per-replica estimators (bead averages), eV except t_centroid (K).
 * k_prim: primitive, k_vir: virial, k_cvir: centroid-virial kinetic energy (S:E1-E3);
 * v_pot: bead-averaged potential for kinds 1-2, NaN for the GFN (it has no energy). */
typedef struct {
    double k_prim, k_vir, k_cvir, v_pot, t_centroid;
} pimd_estimators_t;

/* Bytes of DEVICE workspace pimd_create needs for these sizes.  `out` is HOST. */
int pimd_workspace_bytes(int n_atoms, int n_replicas, int P, const double box[3], const pimd_net_params *net,
                         size_t *out);

/*
 * Creates a context (system + potential + NMPIMD integrator).
 *   species      HOST  [N]      type index 0..S-1
 *   masses_amu   HOST  [S]      mass per type
 *   positions    HOST  [R][N][3] A; every bead of replica r starts here (S:N5)
 *   box          HOST  [3]      orthorhombic edge lengths, {0,0,0} = non-periodic
 *   P, T_kelvin, dt_fs          beads, temperature, time step
 *   gamma_centroid_per_ps       PILE-L centroid friction; < 0 switches the thermostat off (NVE)
 *   seed                        Philox4x32-10 key (S:N4)
 *   d_workspace  DEVICE         caller-allocated (e.g. a torch tensor), >= pimd_workspace_bytes,
 *                               256-byte aligned; the library never allocates or frees device memory
 *   cuda_stream                 cudaStream_t on which every kernel and copy is enqueued
 * Host inputs are copied (synchronously) before the call returns.  Initial momenta are drawn
 * on the device per normal mode (S:N5); forces are evaluated lazily by the first call that
 * needs them.
 */
int pimd_create(pimd_ctx **out, int n_atoms, int n_replicas, const int32_t *species, const double *masses_amu,
                const double *positions, const double box[3], int P, double T_kelvin, double dt_fs,
                double gamma_centroid_per_ps, uint64_t seed, const pimd_net_params *net, void *d_workspace,
                size_t workspace_bytes, void *cuda_stream);

/* Integrator variant, to be chosen before the first step (the initial momenta are redrawn in the chosen representation, S:N5).
 *   transform   0 normal modes (default; S:N2)
 *               1 staging transformation ("the normal mode or staging transformation is employed to decouple the
 *                 evolution of individual beads"): u_0 = q_0, u_j = q_j - (j q_{j+1} + q_0)/(j+1); staging masses m (j+1)/j,
 *                 every staging mode j >= 1 is propagated exactly at w_P, u_0 moves freely
 *               2 primitive ("inter-bead harmonic coupling potentials are incorporated as pluggable energy terms"):
 *                 no transformation; the ring springs are explicit forces in the B half-steps, beads fly freely in A
 *   thermostat  0 PILE-L: Langevin on every mode, friction gamma on the free mode, 2 w_k on the others
 *                 (with transform 2: white-noise Langevin with gamma on every bead)
 *               1 PILE-G: the free mode of all atoms of a replica is rescaled by one stochastic factor (global velocity
 *                 rescaling with time constant 1/gamma); the other modes as PILE-L.  Not available with transform 2.
 * Returns PIMD_ERR_ARG after the first step or for an unsupported combination.  Synchronises. */
int pimd_set_integrator(pimd_ctx *ctx, int transform, int thermostat);

/* n steps of O(dt/2) B(dt/2) A(dt) [neighbour list, forces] B(dt/2) O(dt/2) (S:N3).
 * Asynchronous on the stream; no host synchronisation. */
int pimd_step(pimd_ctx *ctx, int n);

/* Rebuilds the neighbour list and evaluates the forces at the current positions.
 * d_out DEVICE float [R][P][N][3] eV/A.  Asynchronous. */
int pimd_forces(pimd_ctx *ctx, float *d_out);

/* h_out HOST [R].  Synchronises the stream. */
int pimd_estimators(pimd_ctx *ctx, pimd_estimators_t *h_out);

/* State access for parity tests, checkpoint/resume and a host-driven loop.  d_q, d_p double [R][P][N][3]
 * (A, amu*A/fs * 103.6426965268 i.e. eV fs/A), in DEVICE memory or in PAGE-LOCKED HOST memory (the copies are
 * cudaMemcpyAsync with cudaMemcpyDefault on the context's stream; pageable host memory is not supported: the caller
 * could not know when an asynchronous copy has read it); either may be NULL.  `step` HOST.
 * pimd_get_state synchronises (the buffers are the caller's when it returns); pimd_set_state is asynchronous -- the
 * source buffers must stay untouched until the stream has passed the call (pimd_sync, or any synchronising call) --
 * and invalidates the cached forces. */
int pimd_get_state(pimd_ctx *ctx, double *d_q, double *d_p, int64_t *step);
int pimd_set_state(pimd_ctx *ctx, const double *d_q, const double *d_p, int64_t step);

/* The cached forces F(q) belong to a checkpoint too: a resume that restores them skips the force evaluation
 * pimd_set_state would otherwise trigger (same trajectory bit for bit either way; S:N3 step 4 recomputes F from q).
 *   pimd_get_forces_cached  d_F double [R][P][N][3] eV/A (device or page-locked host, as above), the forces at the current q
 *                           (evaluated if stale);
 *                           asynchronous.
 *   pimd_set_forces_cached  d_F device or page-locked host; the caller asserts that d_F = F(q) for the q given to the last pimd_set_state.
 *                           Asynchronous; marks the cached forces valid. */
int pimd_get_forces_cached(pimd_ctx *ctx, double *d_F);
int pimd_set_forces_cached(pimd_ctx *ctx, const double *d_F);

/* Builds the neighbour list at the current positions and exports it as CSR over all rows.
 *   d_row_ptr DEVICE int32 [R*P*N + 1]; d_col DEVICE int32 [col_capacity] holds the atom index j
 *   (0..N-1, within the bead-system of the row), ascending within each row (S:L1);
 *   h_n_pairs HOST.  Synchronises. */
int pimd_nlist(pimd_ctx *ctx, int32_t *d_row_ptr, int32_t *d_col, int64_t col_capacity, int64_t *h_n_pairs);

/* Neighbour-list reuse (the paper fixes only the cutoff, so any list that yields the forces of the exact-r_cut list is
 * admissible): candidates within r_cut + skin are collected by the cell-list pass and kept until some atom has moved by skin/2
 * or more (checked on the device every step, no host synchronisation); every step the exact list d^2 < r_cut^2 (S:L3) is
 * filtered from them, so pimd_nlist and the forces are identical for every skin.  skin in A; 0 = cell-list pass every step.
 * Default: 0 (pays only when atoms move by less than skin/2 over many steps).  PIMD_ERR_ARG unless every periodic box edge
 * >= 2 (r_cut + skin).
 * Asynchronous. */
int pimd_set_nlist_skin(pimd_ctx *ctx, double skin);
/* Number of cell-list passes (candidate-list rebuilds) so far.  h_count HOST.  Synchronises. */
int pimd_nlist_rebuilds(pimd_ctx *ctx, int64_t *h_count);

/* Well-tempered metadynamics with the paper's collective variables.  One bias V_G(s) per replica; the CV is evaluated
 * on every bead and every bead feels F = -dV_G/ds(s_k) grad s(q_k), added to the forces of the potential.  Every
 * `deposit_every` steps (100; 0.05 ps) one Gaussian per bead is deposited at the bead's CV value, width sigma
 * (P:L140, 2 sigma read as 2 sigma^2), height (height_eV / P) exp(-V_G(s_k) / (k_B T (bias_factor - 1))) with the bias before the event.
 *   cv 1  s_dimer = d(O1,H1) - d(O2,H1) + d(O4,H2) - d(O3,H2); atoms6 HOST = indices of O1, H1, O2, O4, H2, O3
 *   cv 2  s_water = (1/N) sum_i sum_j f_i f_j sin(Q R_ij)/(Q R_ij) (all ordered pairs, i = j included, minimum image);
 *         f_species HOST [S] scattering factor per type, Q in 1/A (4 pi sin(11.95 deg) / 1.54 A)
 * The workspace holds up to 16384 Gaussians per replica (further depositions are dropped).  Steps run with plain launches.
 *   pimd_metad_cv          d_s DEVICE double [R][P], d_grad DEVICE double [R][P][N][3] (either may be NULL): CV and its gradient at the
 *                          current positions.  Asynchronous.
 *   pimd_metad_gaussians   HOST copies of the centres and heights of one replica (first `cap`), *h_n = number deposited.  Synchronises.
 *   pimd_metad_deposit_now one deposition event at the current positions (tests, restart). */
int pimd_metad_enable(pimd_ctx *ctx, int cv, const int32_t *atoms6, const double *f_species, double Q, double sigma,
                      double height_eV, double bias_factor, int deposit_every);
int pimd_metad_cv(pimd_ctx *ctx, double *d_s, double *d_grad);
int pimd_metad_gaussians(pimd_ctx *ctx, int replica, double *h_centres, double *h_heights, int cap, int *h_n);
int pimd_metad_deposit_now(pimd_ctx *ctx);

/* The Debye collective variable (cv 2 above: P:L215) WITHOUT a context and WITHOUT any allocation: for callers that
 * cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  Same sum, block
 * partition and summation order as pimd_metad_cv (bit-identical results); its per-block partial sums live in a fixed 128 KB
 * device array inside the library (held by every GPU that loads the library until the process exits).
 *   d_q        DEVICE double [n_systems][n_atoms][3] A;  d_species DEVICE int32 [n_atoms] (type index 0..n_species-1)
 *   box        HOST [3] A, all > 0 (orthorhombic, minimum image) or all 0 (open);  f_species HOST [n_species];  Q in 1/A, > 0
 *   d_s        DEVICE double [n_systems] out;  d_grad DEVICE double [n_systems][n_atoms][3] out, or NULL
 * Limits: n_systems <= 256, n_atoms <= 8192, n_species <= 16; larger sizes return PIMD_ERR_ARG.  Asynchronous on `cuda_stream`
 * (two kernel launches; no cudaMalloc, cudaFree or allocating library call).  Every call shares the scratch array: calls that
 * OVERLAP on the GPU (different streams, parallel graph branches) race on it and must be serialised by the caller.  The
 * array keeps the last call's contents; nothing in it needs clearing (each call writes every entry it reads). */
int pimd_debye_cv_static(const double *d_q, const int32_t *d_species, int n_atoms, int n_systems, const double box[3],
                         const double *f_species, int n_species, double Q, double *d_s, double *d_grad, void *cuda_stream);

/* Waits for the stream and returns any latched device error. */
int pimd_sync(pimd_ctx *ctx);

/* Per-kernel-class device timing with CUDA events recorded on the context's stream around each launch
 * (classes: 0 pimd_nm, 1 nlist, 2 gfn.pair message pass, 3 gfn.node, 4 gfn.head, 5 other).
 * pimd_profile(ctx, 1) starts (and clears) recording, pimd_profile(ctx, 0) stops it.
 * pimd_profile_read synchronises and writes, per class, the summed milliseconds and the number of
 * timed launches into HOST arrays of length 6. */
#define PIMD_PROF_CLASSES 6
int pimd_profile(pimd_ctx *ctx, int enable);
int pimd_profile_read(pimd_ctx *ctx, double *h_ms, int64_t *h_launches);

/* Measurement helper (no context needed): the FP32 fused-multiply-add rate of the current device in TFLOP/s, measured with a
 * kernel of independent FMA chains (best of six launches, CUDA events on `cuda_stream`).  It is the denominator of the "alu"
 * roofline of the fp32 pair kernel (the benchmark must measure it).  h_tflops HOST.  Synchronises. */
int pimd_measure_fp32_fma_tflops(void *cuda_stream, double *h_tflops);

/* Number of kernels the library has launched on this context so far (HOST counter). */
int64_t pimd_launch_count(const pimd_ctx *ctx);

const char *pimd_last_error(void);
void pimd_destroy(pimd_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* PIMD_B200_H */
