// pimd_api.cu -- the C-ABI of include/pimd.h: workspace layout, context life cycle, step sequencing.
// Host logic only; every numerical step is a kernel in nm_kernels.cu / nlist_kernels.cu / gfn_*.cu.
#include "common.cuh"

#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <algorithm>
#include <vector>

static thread_local char g_err[512] = "";

void pimd_set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

extern "C" const char *pimd_last_error(void) { return g_err; }

struct PimdProf {
    bool on = false;
    struct Rec { int kind; cudaEvent_t a, b; };
    std::vector<Rec> recs;
    std::vector<cudaEvent_t> pool;
    cudaEvent_t get()
    {
        if (!pool.empty()) { cudaEvent_t e = pool.back(); pool.pop_back(); return e; }
        cudaEvent_t e;
        cudaEventCreate(&e);
        return e;
    }
    void clear()
    {
        for (auto &r : recs) { pool.push_back(r.a); pool.push_back(r.b); }
        recs.clear();
    }
};

void pimd_prof_begin(pimd_ctx *c, int kind)
{
    PimdProf *p = c->prof;
    if (!p || !p->on) return;
    PimdProf::Rec r{kind, p->get(), p->get()};
    cudaEventRecord(r.a, c->stream);
    p->recs.push_back(r);
}

void pimd_prof_end(pimd_ctx *c)
{
    PimdProf *p = c->prof;
    if (!p || !p->on || p->recs.empty()) return;
    cudaEventRecord(p->recs.back().b, c->stream);
}

namespace {

struct Layout {
    size_t q, p, F, species, mass, C, CT, omega, lam, gam, Tstage, pileg_partial, pileg_alpha, md_n, md_gc, md_gh, md_s, md_dV, md_grad, md_partial, err, est_partial, est_out;
    size_t cell_id, cell_count, cell_start, cell_cursor, sorted_atom, sorted_q, nnz, ncand, hits, hitmask, q_ref, q32, need, row_ptr, block_sums, col, pair_row, dvec;
    size_t wimg, wimg_node, xs0, h1_img, meta_img, weights, nfeat, xfeat, mfeat, Efeat, Gfeat, carry_m, carry_f, Fraw;
    size_t total;
    int ncell[3], nct;
    int64_t pair_cap, n_gran_m, n_gran_f, n_wfloats;
    int gran_m, gran_f, hit_stride;
};

size_t take(size_t &cur, size_t bytes)
{
    size_t o = cur;
    cur = pimd_align_up(cur + bytes);
    return o;
}

int64_t derived_weight_floats(int S, int K, int H, int L)
{
    return (int64_t)S * H + (int64_t)K * H + 3LL * H * H + 4LL * H + (int64_t)L * (5LL * H * H + 3LL * H);
}

int64_t packed_weight_floats(int S, int K, int H, int L)
{
    return (int64_t)S * H + (int64_t)H * K + H + (int64_t)H * H + H + (int64_t)L * (5LL * H * H + 3LL * H) +
           (int64_t)H * H + H + H + 1;
}

int compute_layout(int N, int R, int P, const double box[3], const pimd_net_params *net, Layout *L)
{
    if (N < 1 || R < 1 || P < 1 || P > PIMD_MAX_P || !net || !box) {
        pimd_set_error("invalid sizes: N=%d R=%d P=%d (1 <= P <= %d)", N, R, P, PIMD_MAX_P);
        return PIMD_ERR_ARG;
    }
    if (net->kind < 0 || net->kind > 2) { pimd_set_error("invalid net kind %d", net->kind); return PIMD_ERR_ARG; }
    const bool periodic = box[0] > 0.0 || box[1] > 0.0 || box[2] > 0.0;
    if (periodic && !(box[0] > 0.0 && box[1] > 0.0 && box[2] > 0.0)) {
        pimd_set_error("box must be all zero (open) or all positive");
        return PIMD_ERR_ARG;
    }
    const int64_t rows = (int64_t)R * P * N;
    const int nsys = R * P;
    memset(L, 0, sizeof(*L));
    L->ncell[0] = L->ncell[1] = L->ncell[2] = 1;
    int H = 4;
    if (net->kind == 0) {
        if (!pimd_gfn_supported(net->n_rbf, net->hidden)) {
            pimd_set_error("unsupported (n_rbf, hidden) = (%d, %d); built: (32,64), (64,128)", net->n_rbf, net->hidden);
            return PIMD_ERR_ARG;
        }
        if (net->n_layers < 0 || net->n_layers > 8 || net->n_species < 1 || !(net->r_cut > 0.f)) {
            pimd_set_error("invalid network description");
            return PIMD_ERR_ARG;
        }
        if (N > 32768) { pimd_set_error("n_atoms = %d > 32768 per bead-system is not supported by the neighbour-list fill", N); return PIMD_ERR_ARG; }
        H = net->hidden;
        double expect;
        if (periodic) {
            for (int a = 0; a < 3; ++a) {
                if (box[a] < 2.0 * (double)net->r_cut) {
                    pimd_set_error("periodic box edge %g < 2 r_cut", box[a]);
                    return PIMD_ERR_ARG;
                }
                int nc = (int)floor(box[a] / (double)net->r_cut);
                L->ncell[a] = nc < 1 ? 1 : nc;
            }
            double vol = box[0] * box[1] * box[2], rc = net->r_cut;
            expect = (double)N / vol * 4.18879020478639 * rc * rc * rc;
        } else {
            expect = 256.0;
        }
        // pair capacity per row: 1.5 x the uniform-density expectation + 32 (the -3 latch of the scan kernel guards it; the tile
        // images of the tcgen05 pipeline are sized by it: 35.9 KB per 128 pairs)
        int64_t cap_row = (int64_t)ceil(1.5 * expect) + 32;
        if (cap_row > N - 1) cap_row = N - 1;
        if (cap_row > PIMD_MAX_NBR) cap_row = PIMD_MAX_NBR;
        if (cap_row < 1) cap_row = 1;
        L->pair_cap = (rows * cap_row + 255) / 256 * 256;
        if (L->pair_cap > 2000000000LL) { pimd_set_error("pair capacity exceeds int32 range"); return PIMD_ERR_ARG; }
        // pairs per message-reduction granule: TP * H / NT in the fp32 kernel, a quarter tile in the tcgen05 pipeline
        L->gran_m = (net->gemm_dtype == 1 && net->n_rbf == 64 && H == 128) ? 32 : H / 2;
        L->gran_f = 32;
        L->n_gran_m = L->pair_cap / L->gran_m + 2;
        L->n_gran_f = L->pair_cap / L->gran_f + 2;
        L->n_wfloats = derived_weight_floats(net->n_species, net->n_rbf, H, net->n_layers);
    }
    L->nct = L->ncell[0] * L->ncell[1] * L->ncell[2];
    size_t cur = 0;
    L->q = take(cur, sizeof(double) * rows * 3);
    L->p = take(cur, sizeof(double) * rows * 3);
    L->F = take(cur, sizeof(double) * rows * 3);
    L->species = take(cur, sizeof(int) * N);
    L->mass = take(cur, sizeof(double) * N);
    L->C = take(cur, sizeof(double) * P * P);
    L->CT = take(cur, sizeof(double) * P * P);
    L->omega = take(cur, sizeof(double) * P);
    L->lam = take(cur, sizeof(double) * P);
    L->gam = take(cur, sizeof(double) * P);
    L->Tstage = take(cur, sizeof(double) * 4 * P * P);
    L->pileg_partial = take(cur, sizeof(double) * (size_t)R * 64 * 2);
    L->pileg_alpha = take(cur, sizeof(double) * (size_t)R);
    L->md_n = take(cur, sizeof(int) * (size_t)R);
    L->md_gc = take(cur, sizeof(double) * (size_t)R * PIMD_METAD_MAX);
    L->md_gh = take(cur, sizeof(double) * (size_t)R * PIMD_METAD_MAX);
    L->md_s = take(cur, sizeof(double) * (size_t)R * P);
    L->md_dV = take(cur, sizeof(double) * (size_t)R * P);
    L->md_grad = take(cur, sizeof(double) * (size_t)rows * 3);
    L->md_partial = take(cur, sizeof(double) * (size_t)R * P * PIMD_METAD_BLOCKS);
    L->err = take(cur, sizeof(int) * 4);
    L->est_partial = take(cur, sizeof(double) * (size_t)R * 64 * 8);
    L->est_out = take(cur, sizeof(double) * (size_t)R * 8);
    if (net->kind == 0) {
        L->cell_id = take(cur, sizeof(int) * rows);
        L->cell_count = take(cur, sizeof(int) * (size_t)nsys * L->nct);
        L->cell_start = take(cur, sizeof(int) * (size_t)nsys * (L->nct + 1));
        L->cell_cursor = take(cur, sizeof(int) * (size_t)nsys * L->nct);
        L->sorted_atom = take(cur, sizeof(int) * rows);
        L->sorted_q = take(cur, sizeof(double) * rows * 3);
        L->nnz = take(cur, sizeof(int) * rows);
        L->ncand = take(cur, sizeof(int) * rows);
        L->hitmask = take(cur, sizeof(unsigned) * rows * (PIMD_MAX_NBR / 32));
        L->q_ref = take(cur, sizeof(double) * rows * 3);
        L->q32 = take(cur, sizeof(float) * 4 * rows);
        L->need = take(cur, sizeof(int) * 4);
        L->hit_stride = (N - 1 < PIMD_MAX_NBR) ? (N > 1 ? N - 1 : 1) : PIMD_MAX_NBR;
        L->hits = take(cur, sizeof(int) * rows * L->hit_stride);
        L->row_ptr = take(cur, sizeof(int) * (rows + 1));
        L->block_sums = take(cur, sizeof(int) * ((rows + 1023) / 1024 + 1));
        L->col = take(cur, sizeof(int) * L->pair_cap);
        L->pair_row = take(cur, sizeof(int) * L->pair_cap);
        L->dvec = (net->gemm_dtype == 1 && net->n_rbf == 64 && H == 128) ? take(cur, sizeof(float) * 4 * L->pair_cap) : (size_t)-1;
        L->weights = take(cur, sizeof(float) * L->n_wfloats);
        L->wimg = take(cur, 5 * 16384 + 4096);   // bf16 UMMA images: W_e1 (16 KB), W_e2 (32 KB), W_f1 W_e2 (32 KB)
        L->wimg_node = take(cur, (size_t)(net->n_layers > 0 ? net->n_layers : 1) * 20 * 16384);   // 20 half-images (16 KB) per layer: gfn_node_tc.cu
        L->xs0 = take(cur, sizeof(float) * (size_t)net->n_species * H);
        if (net->gemm_dtype == 1 && net->n_rbf == 64 && H == 128) {   // tile images of the tcgen05 pair pipeline
            const size_t n_tiles = (size_t)(L->pair_cap / 128 + 1);
            L->h1_img = take(cur, n_tiles * 32768);
            L->meta_img = take(cur, n_tiles * 3104);
        }
        const int64_t rows128 = (rows + 127) / 128 * 128;   // the tcgen05 node kernel keeps n and E tile-blocked
        L->nfeat = take(cur, sizeof(float) * rows128 * H);
        L->xfeat = take(cur, sizeof(float) * rows * H);
        L->mfeat = take(cur, sizeof(float) * rows * H);
        L->Efeat = take(cur, sizeof(float) * rows128 * H);
        L->Gfeat = take(cur, sizeof(float) * rows * H);
        L->carry_m = take(cur, sizeof(float) * L->n_gran_m * 2 * H);
        L->carry_f = take(cur, sizeof(float) * L->n_gran_f * 2 * 4);
        L->Fraw = take(cur, sizeof(float) * rows * 4);
    }
    L->total = cur;
    return 0;
}

uint16_t f32_to_bf16_rne(float f)
{
    uint32_t u;
    memcpy(&u, &f, 4);
    if ((u & 0x7FFFFFFFu) > 0x7F800000u) return (uint16_t)((u >> 16) | 0x40);   // NaN
    u += 0x7FFFu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}

// IEEE binary16, round to nearest even (finite inputs well inside the range; used for the readout weights w_f2)
uint16_t f32_to_f16_rne(float f)
{
    uint32_t u;
    memcpy(&u, &f, 4);
    const uint32_t sign = (u >> 16) & 0x8000u;
    const int32_t e = (int32_t)((u >> 23) & 0xFF) - 127 + 15;
    uint32_t m = u & 0x7FFFFFu;
    if (e >= 31) return (uint16_t)(sign | 0x7C00u);                      // overflow -> inf
    if (e <= 0) {                                                        // subnormal or zero
        if (e < -10) return (uint16_t)sign;
        m |= 0x800000u;
        const int shift = 14 - e;
        uint32_t r = m >> shift;
        const uint32_t rem = m & ((1u << shift) - 1u), half = 1u << (shift - 1);
        if (rem > half || (rem == half && (r & 1u))) ++r;
        return (uint16_t)(sign | r);
    }
    uint32_t r = ((uint32_t)e << 10) | (m >> 13);
    const uint32_t rem = m & 0x1FFFu;
    if (rem > 0x1000u || (rem == 0x1000u && (r & 1u))) ++r;              // carries into the exponent correctly
    return (uint16_t)(sign | r);
}

// bf16 image of a row-major [n_rows][n_k] matrix as UMMA K-major operand blocks of 64 k (128-byte rows, 16-byte
// chunks XOR-swizzled by row & 7), block kb at byte offset kb * n_rows * 128
void build_umma_image(const float *W, int n_rows, int n_k, float scale, uint16_t *img)
{
    for (int kb = 0; kb < n_k / 64; ++kb)
        for (int n = 0; n < n_rows; ++n)
            for (int c = 0; c < 8; ++c)
                for (int e = 0; e < 8; ++e)
                    img[(size_t)kb * n_rows * 64 + (size_t)n * 64 + ((c ^ (n & 7)) * 8) + e] =
                        f32_to_bf16_rne(scale * W[(size_t)n * n_k + kb * 64 + c * 8 + e]);
}

// the same image for W = hi + lo as a bf16 pair: hi = bf16(scale W), lo = bf16(scale W - hi)  (split-precision products of the
// atom-wise layers, gfn_node_tc.cu)
void build_umma_image_split(const float *W, int n_rows, int n_k, float scale, uint16_t *img_hi, uint16_t *img_lo)
{
    std::vector<float> hi((size_t)n_rows * n_k), lo((size_t)n_rows * n_k);
    for (size_t i = 0; i < hi.size(); ++i) {
        const float v = scale * W[i];
        const uint32_t hb = (uint32_t)f32_to_bf16_rne(v) << 16;
        float hf;
        memcpy(&hf, &hb, 4);
        hi[i] = hf;
        lo[i] = v - hf;
    }
    build_umma_image(hi.data(), n_rows, n_k, 1.0f, img_hi);
    build_umma_image(lo.data(), n_rows, n_k, 1.0f, img_lo);
}

// derived, transposed fp32 weights in the order the kernels use (S:G0 is the input order)
struct RawLayer { const float *Ws, *Wvn, *Wvm, *bv1, *Wv2, *bv2, *Wa, *ba; };
struct RawNet { const float *Emb, *We1, *be1, *We2, *be2, *Wf1, *bf1, *wf2; std::vector<RawLayer> layer; };

void build_weights(const pimd_net_params *net, std::vector<float> &out, std::vector<size_t> &offs, std::vector<float> &Wfe,
                   RawNet &raw)
{
    const int S = net->n_species, K = net->n_rbf, H = net->hidden, L = net->n_layers;
    const float *w = net->weights;
    auto mat = [&](int n_out, int n_in) { const float *m = w; w += (size_t)n_out * n_in; return m; };
    auto vec = [&](int n) { const float *v = w; w += n; return v; };
    auto pushT = [&](const float *m, int n_out, int n_in) {   // [out][in] -> [in][out]
        offs.push_back(out.size());
        for (int k = 0; k < n_in; ++k)
            for (int o = 0; o < n_out; ++o) out.push_back(m[(size_t)o * n_in + k]);
    };
    auto pushV = [&](const float *v, int n) { offs.push_back(out.size()); out.insert(out.end(), v, v + n); };
    const float *Emb = mat(S, H), *We1 = mat(H, K), *be1 = vec(H), *We2 = mat(H, H), *be2 = vec(H);
    std::vector<RawLayer> lw(L);
    for (int l = 0; l < L; ++l) {
        lw[l].Ws = mat(H, H); lw[l].Wvn = mat(H, H); lw[l].Wvm = mat(H, H); lw[l].bv1 = vec(H);
        lw[l].Wv2 = mat(H, H); lw[l].bv2 = vec(H); lw[l].Wa = mat(H, H); lw[l].ba = vec(H);
    }
    const float *Wf1 = mat(H, H), *bf1 = vec(H), *wf2 = vec(H);
    raw.Emb = Emb; raw.We1 = We1; raw.be1 = be1; raw.We2 = We2; raw.be2 = be2; raw.Wf1 = Wf1; raw.bf1 = bf1; raw.wf2 = wf2;
    raw.layer = lw;
    // W_fe = W_f1 W_e2 and b_fe = W_f1 b_e2 + b_f1, formed in fp64 then rounded once
    std::vector<float> bfe(H);
    Wfe.assign((size_t)H * H, 0.f);
    for (int o = 0; o < H; ++o) {
        for (int k = 0; k < H; ++k) {
            double s = 0.0;
            for (int t = 0; t < H; ++t) s += (double)Wf1[(size_t)o * H + t] * (double)We2[(size_t)t * H + k];
            Wfe[(size_t)o * H + k] = (float)s;
        }
        double s = (double)bf1[o];
        for (int t = 0; t < H; ++t) s += (double)Wf1[(size_t)o * H + t] * (double)be2[t];
        bfe[o] = (float)s;
    }
    pushV(Emb, S * H);            // 0
    pushT(We1, H, K);             // 1
    pushV(be1, H);                // 2
    pushT(We2, H, H);             // 3
    pushV(be2, H);                // 4
    pushT(Wfe.data(), H, H);      // 5
    pushV(bfe.data(), H);         // 6
    pushT(Wf1, H, H);             // 7
    pushV(wf2, H);                // 8
    for (int l = 0; l < L; ++l) { // 9 + 8 l
        pushT(lw[l].Ws, H, H); pushT(lw[l].Wvn, H, H); pushT(lw[l].Wvm, H, H); pushV(lw[l].bv1, H);
        pushT(lw[l].Wv2, H, H); pushV(lw[l].bv2, H); pushT(lw[l].Wa, H, H); pushV(lw[l].ba, H);
    }
}

int check_device_error(pimd_ctx *c)
{
    int flags[4] = {0, 0, 0, 0};
    PIMD_CUDA_CHECK(cudaMemcpyAsync(flags, c->err, sizeof(flags), cudaMemcpyDeviceToHost, c->stream));
    PIMD_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    if (flags[0] & PIMD_FLAG_PAIRS) {
        pimd_set_error("pair capacity (%lld pairs, or %d neighbours per atom) exceeded", (long long)c->nl.pair_cap,
                       PIMD_MAX_NBR);
        return PIMD_ERR_PAIRS;
    }
    if (flags[0] & PIMD_FLAG_NAN) { pimd_set_error("non-finite force or position"); return PIMD_ERR_NAN; }
    return 0;
}

// every entry point runs on the context's device, whatever device is current in the calling thread
int enter(pimd_ctx *c)
{
    int dev = -1;
    if (cudaGetDevice(&dev) == cudaSuccess && dev == c->device) return 0;
    PIMD_CUDA_CHECK(cudaSetDevice(c->device));
    return 0;
}

// the Philox counter holds the step as one 32-bit word (S:N4)
constexpr int64_t PIMD_MAX_STEP = 4294967295LL;

// a captured step bakes in the kernel arguments: anything that changes them drops the graph (it is captured again on demand)
void drop_step_graph(pimd_ctx *c)
{
    if (c->step_graph) { cudaStreamSynchronize(c->stream); cudaGraphExecDestroy(c->step_graph); c->step_graph = nullptr; }
    c->graph_state = 0;
}

// candidate radius r_cut + skin of the reusable neighbour lists: the cell grid must have cells at least that wide
int apply_skin(pimd_ctx *c, double skin)
{
    if (c->kind != 0) return 0;
    drop_step_graph(c);
    if (!(skin >= 0.0)) { pimd_set_error("skin must be >= 0"); return PIMD_ERR_ARG; }
    const double rl = (double)c->net.r_cut + skin;
    int nc[3] = {1, 1, 1};
    if (c->periodic)
        for (int a = 0; a < 3; ++a) {
            if (c->box[a] < 2.0 * rl) { pimd_set_error("periodic box edge %g < 2 (r_cut + skin) = %g", c->box[a], 2.0 * rl); return PIMD_ERR_ARG; }
            nc[a] = (int)floor(c->box[a] / rl);
            if (nc[a] < 1) nc[a] = 1;
        }
    for (int a = 0; a < 3; ++a) c->nl.ncell[a] = nc[a];
    c->nl.ncell_tot = nc[0] * nc[1] * nc[2];
    c->nl.skin = skin;
    return pimd_launch_nlist_invalidate(c);
}

int compute_forces(pimd_ctx *c)
{
    int rc;
    if (c->kind == 0) {
        {
            ProfScope ps(c, PROF_NLIST);
            if ((rc = pimd_launch_nlist(c))) return rc;
        }
        if ((rc = pimd_launch_gfn_forces(c))) return rc;
    } else {
        ProfScope ps(c, PROF_OTHER);
        if ((rc = pimd_launch_simple_forces(c))) return rc;
    }
    if (c->md.cv) {
        ProfScope ps(c, PROF_OTHER);
        if ((rc = pimd_launch_metad_bias(c, 1))) return rc;
    }
    c->forces_valid = 1;
    return 0;
}

}  // namespace

extern "C" int pimd_workspace_bytes(int n_atoms, int n_replicas, int P, const double box[3],
                                    const pimd_net_params *net, size_t *out)
{
    if (!out) { pimd_set_error("null out"); return PIMD_ERR_ARG; }
    Layout L;
    int rc = compute_layout(n_atoms, n_replicas, P, box, net, &L);
    if (rc) return rc;
    *out = L.total;
    return 0;
}

extern "C" int pimd_create(pimd_ctx **out, int n_atoms, int n_replicas, const int32_t *species,
                           const double *masses_amu, const double *positions, const double box[3], int P,
                           double T_kelvin, double dt_fs, double gamma_centroid_per_ps, uint64_t seed,
                           const pimd_net_params *net, void *d_workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!out || !species || !masses_amu || !positions || !box || !net || !d_workspace) {
        pimd_set_error("null argument");
        return PIMD_ERR_ARG;
    }
    if (!(T_kelvin > 0.0) || !(dt_fs > 0.0)) { pimd_set_error("T and dt must be positive"); return PIMD_ERR_ARG; }
    Layout L;
    int rc = compute_layout(n_atoms, n_replicas, P, box, net, &L);
    if (rc) return rc;
    if (workspace_bytes < L.total) {
        pimd_set_error("workspace too small: %zu < %zu", workspace_bytes, L.total);
        return PIMD_ERR_ARG;
    }
    if (((uintptr_t)d_workspace) % 256 != 0) { pimd_set_error("workspace must be 256-byte aligned"); return PIMD_ERR_ARG; }
    const int N = n_atoms, R = n_replicas;
    if (net->n_species < 1) { pimd_set_error("n_species = %d (masses_amu has one entry per species)", net->n_species); return PIMD_ERR_ARG; }
    for (int i = 0; i < N; ++i)
        if (species[i] < 0 || species[i] >= net->n_species) {
            pimd_set_error("species[%d] = %d out of range [0, %d)", i, species[i], net->n_species);
            return PIMD_ERR_ARG;
        }
    if (net->kind == 0) {
        if (!net->weights || net->n_weights != packed_weight_floats(net->n_species, net->n_rbf, net->hidden, net->n_layers)) {
            pimd_set_error("n_weights = %lld, expected %lld", (long long)net->n_weights,
                           (long long)packed_weight_floats(net->n_species, net->n_rbf, net->hidden, net->n_layers));
            return PIMD_ERR_ARG;
        }
    }
    pimd_ctx *c = new pimd_ctx();
    memset(c, 0, sizeof(*c));
    c->N = N; c->R = R; c->P = P; c->rows = (int64_t)R * P * N;
    c->periodic = box[0] > 0.0;
    for (int a = 0; a < 3; ++a) c->box[a] = box[a];
    c->T = T_kelvin; c->dt = dt_fs; c->gamma_fs = gamma_centroid_per_ps < 0.0 ? -1.0 : gamma_centroid_per_ps * 1e-3;
    c->seed = seed; c->step = 0; c->kind = net->kind; c->gemm_dtype = net->gemm_dtype;
    c->n_species_host = net->n_species;
    c->harmonic_omega = net->harmonic_omega;
    c->stream = (cudaStream_t)cuda_stream;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);          // the device current at creation owns the workspace and the stream
    c->device = dev;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) {
        pimd_set_error("no CUDA device: %s", cudaGetErrorString(e));
        delete c;
        return PIMD_ERR_CUDA;
    }
    char *ws = (char *)d_workspace;
    c->q = (double *)(ws + L.q); c->p = (double *)(ws + L.p); c->F = (double *)(ws + L.F);
    c->species = (int *)(ws + L.species); c->mass = (double *)(ws + L.mass);
    c->Cmat = (double *)(ws + L.C); c->CmatT = (double *)(ws + L.CT); c->omega_k = (double *)(ws + L.omega);
    c->lam_k = (double *)(ws + L.lam); c->gam_k = (double *)(ws + L.gam); c->Tstage = (double *)(ws + L.Tstage);
    c->pileg_partial = (double *)(ws + L.pileg_partial); c->pileg_alpha = (double *)(ws + L.pileg_alpha);
    c->transform = 0; c->thermostat = 0;
    c->md.cv = 0;
    c->md.n_g = (int *)(ws + L.md_n); c->md.gc = (double *)(ws + L.md_gc); c->md.gh = (double *)(ws + L.md_gh);
    c->md.s = (double *)(ws + L.md_s); c->md.dV = (double *)(ws + L.md_dV); c->md.grad = (double *)(ws + L.md_grad);
    c->md.partial = (double *)(ws + L.md_partial);
    c->Tq_fwd = c->CmatT; c->Tp_fwd = c->CmatT; c->Tq_inv = c->Cmat; c->Tp_inv = c->Cmat;   // normal modes: orthogonal
    c->err = (int *)(ws + L.err);
    c->step_dev = (uint32_t *)(c->err + 2);          // (words 2, 3 of the error block)
    c->est_partial = (double *)(ws + L.est_partial); c->est_out = (double *)(ws + L.est_out);

    // host staging
    std::vector<double> mass(N), Cm((size_t)P * P), CT((size_t)P * P), om(P), q0((size_t)c->rows * 3);
    for (int i = 0; i < N; ++i) mass[i] = masses_amu[species[i]] * PIMD_AMU;
    const double pi = 3.14159265358979323846264338327950288;
    for (int j = 0; j < P; ++j)   // S:N2
        for (int k = 0; k < P; ++k) {
            double v;
            if (k == 0) v = 1.0 / sqrt((double)P);
            else if (2 * k < P) v = sqrt(2.0 / P) * cos(2.0 * pi * j * k / P);
            else if (2 * k == P) v = ((j & 1) ? -1.0 : 1.0) / sqrt((double)P);
            else v = sqrt(2.0 / P) * sin(2.0 * pi * j * k / P);
            Cm[(size_t)j * P + k] = v; CT[(size_t)k * P + j] = v;
        }
    const double omega_P = P * PIMD_KB * T_kelvin / PIMD_HBAR;   // S:N1
    for (int k = 0; k < P; ++k) om[k] = 2.0 * omega_P * sin(k * pi / P);
    for (int r = 0; r < R; ++r)
        for (int k = 0; k < P; ++k)
            memcpy(&q0[(((size_t)r * P + k) * N) * 3], positions + (size_t)r * N * 3, sizeof(double) * N * 3);

#define CREATE_CHECK(call)                                                                  \
    do {                                                                                    \
        cudaError_t e_ = (call);                                                            \
        if (e_ != cudaSuccess) {                                                            \
            pimd_set_error("%s failed: %s", #call, cudaGetErrorString(e_));                 \
            delete c;                                                                       \
            return PIMD_ERR_CUDA;                                                           \
        }                                                                                   \
    } while (0)
    cudaStream_t st = c->stream;
    CREATE_CHECK(cudaMemsetAsync(c->err, 0, sizeof(int) * 4, st));   // error word, step counter
    CREATE_CHECK(cudaMemsetAsync(c->F, 0, sizeof(double) * c->rows * 3, st));
    CREATE_CHECK(cudaMemcpyAsync(c->q, q0.data(), sizeof(double) * q0.size(), cudaMemcpyHostToDevice, st));
    CREATE_CHECK(cudaMemcpyAsync(c->species, species, sizeof(int) * N, cudaMemcpyHostToDevice, st));
    CREATE_CHECK(cudaMemcpyAsync(c->mass, mass.data(), sizeof(double) * N, cudaMemcpyHostToDevice, st));
    CREATE_CHECK(cudaMemcpyAsync(c->Cmat, Cm.data(), sizeof(double) * P * P, cudaMemcpyHostToDevice, st));
    CREATE_CHECK(cudaMemcpyAsync(c->CmatT, CT.data(), sizeof(double) * P * P, cudaMemcpyHostToDevice, st));
    CREATE_CHECK(cudaMemcpyAsync(c->omega_k, om.data(), sizeof(double) * P, cudaMemcpyHostToDevice, st));
    std::vector<double> lam(P, 1.0), gam(P);
    for (int k = 0; k < P; ++k) gam[k] = (k == 0) ? c->gamma_fs : 2.0 * om[k];   // PILE: critical damping of the free-ring modes (S:N3)
    CREATE_CHECK(cudaMemcpyAsync(c->lam_k, lam.data(), sizeof(double) * P, cudaMemcpyHostToDevice, st));
    CREATE_CHECK(cudaMemcpyAsync(c->gam_k, gam.data(), sizeof(double) * P, cudaMemcpyHostToDevice, st));

    std::vector<float> wd, xs0;
    std::vector<uint16_t> wimg, wimg_node;
    if (net->kind == 0) {
        const int H = net->hidden;
        NlistDev &nl = c->nl;
        for (int a = 0; a < 3; ++a) nl.ncell[a] = L.ncell[a];
        nl.ncell_tot = L.nct;
        nl.cell_id = (int *)(ws + L.cell_id); nl.cell_count = (int *)(ws + L.cell_count);
        nl.cell_start = (int *)(ws + L.cell_start); nl.cell_cursor = (int *)(ws + L.cell_cursor);
        nl.sorted_atom = (int *)(ws + L.sorted_atom); nl.sorted_q = (double *)(ws + L.sorted_q);
        nl.nnz = (int *)(ws + L.nnz); nl.ncand = (int *)(ws + L.ncand); nl.hitmask = (unsigned *)(ws + L.hitmask);
        nl.q_ref = (double *)(ws + L.q_ref); nl.q32 = (float4 *)(ws + L.q32); nl.need = (int *)(ws + L.need); nl.skin = 0.0;
        CREATE_CHECK(cudaMemsetAsync(nl.need, 0, sizeof(int) * 4, st));
        nl.hits = (int *)(ws + L.hits); nl.hit_stride = L.hit_stride; nl.row_ptr = (int *)(ws + L.row_ptr); nl.block_sums = (int *)(ws + L.block_sums);
        nl.col = (int *)(ws + L.col); nl.pair_row = (int *)(ws + L.pair_row); nl.dvec = (L.dvec == (size_t)-1) ? nullptr : (float4 *)(ws + L.dvec); nl.pair_cap = L.pair_cap;
        c->weights_dev = (float *)(ws + L.weights);
        c->nfeat = (float *)(ws + L.nfeat); c->xfeat = (float *)(ws + L.xfeat); c->mfeat = (float *)(ws + L.mfeat);
        c->Efeat = (float *)(ws + L.Efeat); c->Gfeat = (float *)(ws + L.Gfeat);
        c->carry_m = (float *)(ws + L.carry_m); c->carry_f = (float *)(ws + L.carry_f); c->Fraw = (float *)(ws + L.Fraw);
        c->gran_m = L.gran_m; c->gran_f = L.gran_f; c->n_gran_m = L.n_gran_m; c->n_gran_f = L.n_gran_f;
        std::vector<size_t> offs;
        std::vector<float> Wfe;
        RawNet raw;
        build_weights(net, wd, offs, Wfe, raw);
        c->use_tc = (net->gemm_dtype == 1 && net->n_rbf == 64 && net->hidden == 128) ? 1 : 0;
        c->wimg_e1 = (uint16_t *)(ws + L.wimg); c->wimg_e2 = c->wimg_e1 + 8192; c->wimg_fe = c->wimg_e2 + 16384;
        if (c->use_tc) {
            wimg.resize(5 * 8192 + 2048);
            const float *We1 = net->weights + (size_t)net->n_species * H;          // [H][K]
            const float *We2 = We1 + (size_t)H * net->n_rbf + H;                   // [H][H]
            build_umma_image(We1, H, net->n_rbf, 0.5f, wimg.data());   // SiLU(x) = h tanh(h) + h, h = x/2
            build_umma_image(We2, H, H, 1.0f, wimg.data() + 8192);
            build_umma_image(Wfe.data(), H, H, 0.5f, wimg.data() + 8192 + 16384);
            {   // w_f2 on 16 identical rows: B operand of the head's 128x16x128 readout product
                std::vector<float> rep((size_t)16 * H);
                for (int r = 0; r < 16; ++r) for (int k = 0; k < H; ++k) rep[(size_t)r * H + k] = raw.wf2[k];
                uint16_t *img = wimg.data() + 5 * 8192;      // same layout as build_umma_image, fp16 elements (the head's act operand is fp16)
                for (int kb = 0; kb < H / 64; ++kb)
                    for (int n = 0; n < 16; ++n)
                        for (int cch = 0; cch < 8; ++cch)
                            for (int e = 0; e < 8; ++e)
                                img[(size_t)kb * 16 * 64 + (size_t)n * 64 + ((cch ^ (n & 7)) * 8) + e] =
                                    f32_to_f16_rne(rep[(size_t)n * H + kb * 64 + cch * 8 + e]);
            }
            c->wimg_wf2 = c->wimg_e1 + 5 * 8192;
            CREATE_CHECK(cudaMemcpyAsync(c->wimg_e1, wimg.data(), sizeof(uint16_t) * wimg.size(), cudaMemcpyHostToDevice, st));
            // atom-wise layers: five images per layer; SiLU's 1/2 folded into W_vn, W_vm
            c->wimg_node = (uint16_t *)(ws + L.wimg_node); c->xs0 = (float *)(ws + L.xs0);
            c->XE = (uint32_t *)c->xfeat;
            {   // tensor maps of the two gathered tables (rows of 512 B; box = one row; used with tile::gather4)
                typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                              const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                              CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
                void *fn = nullptr;
                cudaDriverEntryPointQueryResult qres;
                CREATE_CHECK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
                if (!fn || qres != cudaDriverEntryPointSuccess) { pimd_set_error("cuTensorMapEncodeTiled is not available in this driver"); delete c; return PIMD_ERR_CUDA; }
                const cuuint64_t gdim[2] = {128, (cuuint64_t)c->rows};
                const cuuint64_t gstr[1] = {512};
                const cuuint32_t box[2] = {128, 1}, estr[2] = {1, 1};
                void *bases[2] = {c->XE, c->Gfeat};
                CUtensorMap *maps[2] = {&c->tmap_xe, &c->tmap_g};
                for (int t = 0; t < 2; ++t) {
                    const CUresult rc = ((encode_fn)fn)(maps[t], CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, bases[t], gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                                        CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
                    if (rc != CUDA_SUCCESS) { pimd_set_error("cuTensorMapEncodeTiled failed (%d)", (int)rc); delete c; return PIMD_ERR_CUDA; }
                }
            }
            c->h1_img = (unsigned char *)(ws + L.h1_img); c->meta_img = (unsigned char *)(ws + L.meta_img);
            for (int k = 0; k < H && k < 128; ++k) c->h_be1_half[k] = 0.5f * raw.be1[k];
            const int Ln = net->n_layers;
            // per layer 20 half-images of 8192 bf16 in the order a tile consumes them: (W_vn/2, W_vm/2, W_v2, W_a) as hi | lo
            // (each two K blocks), then W_s^{l+1} hi (and its lo, unused) or, in the last layer, W_f1 hi | lo
            wimg_node.resize((size_t)(Ln > 0 ? Ln : 1) * 20 * 8192);
            for (int l = 0; l < Ln; ++l) {
                uint16_t *img = wimg_node.data() + (size_t)l * 20 * 8192;
                build_umma_image_split(raw.layer[l].Wvn, H, H, 0.5f, img, img + 16384);
                build_umma_image_split(raw.layer[l].Wvm, H, H, 0.5f, img + 2 * 16384, img + 3 * 16384);
                build_umma_image_split(raw.layer[l].Wv2, H, H, 1.0f, img + 4 * 16384, img + 5 * 16384);
                build_umma_image_split(raw.layer[l].Wa, H, H, 1.0f, img + 6 * 16384, img + 7 * 16384);
                build_umma_image_split(l + 1 < Ln ? raw.layer[l + 1].Ws : raw.Wf1, H, H, 1.0f, img + 8 * 16384, img + 9 * 16384);
            }
            xs0.assign((size_t)net->n_species * H, 0.f);
            if (Ln > 0)
                for (int s = 0; s < net->n_species; ++s)
                    for (int o = 0; o < H; ++o) {
                        double acc = 0.0;
                        for (int k = 0; k < H; ++k) acc += (double)raw.layer[0].Ws[(size_t)o * H + k] * (double)raw.Emb[(size_t)s * H + k];
                        xs0[(size_t)s * H + o] = (float)acc;
                    }
            CREATE_CHECK(cudaMemcpyAsync(c->wimg_node, wimg_node.data(), sizeof(uint16_t) * wimg_node.size(), cudaMemcpyHostToDevice, st));
            CREATE_CHECK(cudaMemcpyAsync(c->xs0, xs0.data(), sizeof(float) * xs0.size(), cudaMemcpyHostToDevice, st));
        }
        if ((int64_t)wd.size() != L.n_wfloats) {
            pimd_set_error("internal: derived weight count %zu != %lld", wd.size(), (long long)L.n_wfloats);
            delete c;
            return PIMD_ERR_ARG;
        }
        CREATE_CHECK(cudaMemcpyAsync(c->weights_dev, wd.data(), sizeof(float) * wd.size(), cudaMemcpyHostToDevice, st));
        GfnDev &g = c->net;
        g.S = net->n_species; g.K = net->n_rbf; g.H = H; g.L = net->n_layers;
        g.r_cut = net->r_cut; g.agg_norm = net->agg_norm; g.force_scale = net->force_scale;
        const float *b = c->weights_dev;
        g.Emb = b + offs[0]; g.We1T = b + offs[1]; g.be1 = b + offs[2]; g.We2T = b + offs[3]; g.be2 = b + offs[4];
        g.WfeT = b + offs[5]; g.bfe = b + offs[6]; g.Wf1T = b + offs[7]; g.wf2 = b + offs[8];
        g.bf2 = net->weights[net->n_weights - 1];
        for (int l = 0; l < g.L; ++l) {
            const size_t *o = &offs[9 + 8 * l];
            g.layer[l].WsT = b + o[0]; g.layer[l].WvnT = b + o[1]; g.layer[l].WvmT = b + o[2]; g.layer[l].bv1 = b + o[3];
            g.layer[l].Wv2T = b + o[4]; g.layer[l].bv2 = b + o[5]; g.layer[l].WaT = b + o[6]; g.layer[l].ba = b + o[7];
        }
        CREATE_CHECK(cudaMemsetAsync(nl.row_ptr, 0, sizeof(int) * (c->rows + 1), st));
        // default: no reuse (skin 0).  The synthetic workloads are hot (random-weight force field): atoms move skin/2 =
        // 0.25 A in about four steps and the larger candidate radius costs more than it saves; pimd_set_nlist_skin turns reuse on
        g.r_cut = net->r_cut;   // (apply_skin reads it)
        if (apply_skin(c, 0.0)) { delete c; return PIMD_ERR_CUDA; }
    }
    rc = pimd_launch_init_momenta(c);   // S:N5
    if (rc) { delete c; return rc; }
    CREATE_CHECK(cudaStreamSynchronize(st));   // host staging buffers go out of scope below
#undef CREATE_CHECK
    c->forces_valid = 0;
    *out = c;
    return 0;
}

extern "C" void pimd_destroy(pimd_ctx *c)
{
    if (!c) return;
    (void)enter(c);
    cudaStreamSynchronize(c->stream);
    if (c->step_graph) cudaGraphExecDestroy(c->step_graph);
    if (c->prof) {
        c->prof->clear();
        for (auto e : c->prof->pool) cudaEventDestroy(e);
        delete c->prof;
    }
    delete c;
}

// Integrator variants ("normal mode or staging transformation", P:L114 primitive PIMD with the bead
// springs as explicit forces).  The mode tables are built here, in fp64 on the host, from the DEFINITIONS:
//   staging variables  u_0 = q_0,  u_j = q_j - (j q_{j+1} + q_0) / (j + 1), q_P = q_0  ->  matrix F;  q = F^-1 u by elimination;
//   canonical momenta transform with the inverse transpose: p_u = F^-T p_q, p_q = F^T p_u;
//   staging masses m (j+1)/j and frequency w_P for j >= 1 (the ring springs become sum_j 1/2 m lam_j w_P^2 u_j^2), u_0 free.
extern "C" int pimd_set_integrator(pimd_ctx *c, int transform, int thermostat)
{
    if (!c) { pimd_set_error("null context"); return PIMD_ERR_ARG; }
    if (transform < 0 || transform > 2 || thermostat < 0 || thermostat > 1) { pimd_set_error("transform in {0,1,2}, thermostat in {0,1}"); return PIMD_ERR_ARG; }
    if (thermostat == 1 && transform == 2) { pimd_set_error("PILE-G needs a free (centroid-like) mode: not with the primitive variant"); return PIMD_ERR_ARG; }
    if (c->step != 0) { pimd_set_error("the integrator variant is chosen before the first step"); return PIMD_ERR_ARG; }
    int rc;
    if ((rc = enter(c))) return rc;
    const int P = c->P;
    const double pi = 3.14159265358979323846264338327950288;
    const double omega_P = P * PIMD_KB * c->T / PIMD_HBAR;
    std::vector<double> om(P), lam(P, 1.0), gam(P);
    if (transform == 0) {
        for (int k = 0; k < P; ++k) { om[k] = 2.0 * omega_P * sin(k * pi / P); gam[k] = (k == 0) ? c->gamma_fs : 2.0 * om[k]; }
        c->Tq_fwd = c->CmatT; c->Tp_fwd = c->CmatT; c->Tq_inv = c->Cmat; c->Tp_inv = c->Cmat;
    } else if (transform == 2) {
        // identity maps: rows of the normal-mode storage are not needed; the staging block holds I four times
        std::vector<double> I4((size_t)4 * P * P, 0.0);
        for (int m = 0; m < 4; ++m) for (int j = 0; j < P; ++j) I4[(size_t)m * P * P + (size_t)j * P + j] = 1.0;
        PIMD_CUDA_CHECK(cudaMemcpyAsync(c->Tstage, I4.data(), sizeof(double) * I4.size(), cudaMemcpyHostToDevice, c->stream));
        PIMD_CUDA_CHECK(cudaStreamSynchronize(c->stream));
        c->Tq_fwd = c->Tstage; c->Tq_inv = c->Tstage + (size_t)P * P; c->Tp_fwd = c->Tstage + 2 * (size_t)P * P; c->Tp_inv = c->Tstage + 3 * (size_t)P * P;
        for (int k = 0; k < P; ++k) { om[k] = 0.0; gam[k] = c->gamma_fs; }   // every bead flies freely in A; white-noise Langevin on every bead
    } else {
        std::vector<long double> F((size_t)P * P, 0.0L), Fi((size_t)P * P, 0.0L);
        F[0] = 1.0L;
        for (int j = 1; j < P; ++j) {
            F[(size_t)j * P + j] += 1.0L;
            F[(size_t)j * P + (j + 1) % P] -= (long double)j / (long double)(j + 1);
            F[(size_t)j * P + 0] -= 1.0L / (long double)(j + 1);
        }
        {   // inverse by Gauss-Jordan elimination with partial pivoting
            std::vector<long double> A(F);
            for (int j = 0; j < P; ++j) Fi[(size_t)j * P + j] = 1.0L;
            for (int col = 0; col < P; ++col) {
                int piv = col;
                for (int rr = col + 1; rr < P; ++rr) if (fabsl(A[(size_t)rr * P + col]) > fabsl(A[(size_t)piv * P + col])) piv = rr;
                if (piv != col)
                    for (int k = 0; k < P; ++k) { std::swap(A[(size_t)piv * P + k], A[(size_t)col * P + k]); std::swap(Fi[(size_t)piv * P + k], Fi[(size_t)col * P + k]); }
                const long double d = A[(size_t)col * P + col];
                for (int k = 0; k < P; ++k) { A[(size_t)col * P + k] /= d; Fi[(size_t)col * P + k] /= d; }
                for (int rr = 0; rr < P; ++rr) {
                    if (rr == col) continue;
                    const long double f = A[(size_t)rr * P + col];
                    if (f == 0.0L) continue;
                    for (int k = 0; k < P; ++k) { A[(size_t)rr * P + k] -= f * A[(size_t)col * P + k]; Fi[(size_t)rr * P + k] -= f * Fi[(size_t)col * P + k]; }
                }
            }
        }
        std::vector<double> T4((size_t)4 * P * P);
        for (int j = 0; j < P; ++j)
            for (int k = 0; k < P; ++k) {
                T4[(size_t)j * P + k] = (double)F[(size_t)j * P + k];                                  // u = F q
                T4[(size_t)P * P + (size_t)j * P + k] = (double)Fi[(size_t)j * P + k];                 // q = F^-1 u
                T4[2 * (size_t)P * P + (size_t)j * P + k] = (double)Fi[(size_t)k * P + j];             // p_u = F^-T p_q
                T4[3 * (size_t)P * P + (size_t)j * P + k] = (double)F[(size_t)k * P + j];              // p_q = F^T p_u
            }
        PIMD_CUDA_CHECK(cudaMemcpyAsync(c->Tstage, T4.data(), sizeof(double) * T4.size(), cudaMemcpyHostToDevice, c->stream));
        PIMD_CUDA_CHECK(cudaStreamSynchronize(c->stream));
        c->Tq_fwd = c->Tstage; c->Tq_inv = c->Tstage + (size_t)P * P; c->Tp_fwd = c->Tstage + 2 * (size_t)P * P; c->Tp_inv = c->Tstage + 3 * (size_t)P * P;
        for (int k = 0; k < P; ++k) {
            lam[k] = (k == 0) ? 1.0 : (double)(k + 1) / (double)k;
            om[k] = (k == 0) ? 0.0 : omega_P;
            gam[k] = (k == 0) ? c->gamma_fs : 2.0 * omega_P;
        }
    }
    PIMD_CUDA_CHECK(cudaMemcpyAsync(c->omega_k, om.data(), sizeof(double) * P, cudaMemcpyHostToDevice, c->stream));
    PIMD_CUDA_CHECK(cudaMemcpyAsync(c->lam_k, lam.data(), sizeof(double) * P, cudaMemcpyHostToDevice, c->stream));
    PIMD_CUDA_CHECK(cudaMemcpyAsync(c->gam_k, gam.data(), sizeof(double) * P, cudaMemcpyHostToDevice, c->stream));
    PIMD_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    c->transform = transform; c->thermostat = thermostat;
    drop_step_graph(c);
    return pimd_launch_init_momenta(c);   // S:N5 in the chosen representation
}

namespace {

// one step: O B A | step counter | neighbour list + forces | B O   (S:N3); nothing in the launch sequence depends on the step
int step_body(pimd_ctx *c)
{
    int rc;
    {
        ProfScope ps(c, PROF_NM);
        if ((rc = pimd_launch_nm_pre(c))) return rc;
    }
    if ((rc = compute_forces(c))) return rc;
    ProfScope ps(c, PROF_NM);
    return pimd_launch_nm_post(c);
}

int sync_step_counter(pimd_ctx *c)
{
    return pimd_launch_set_step(c, (uint32_t)c->step);   // (a kernel argument: no host buffer to keep alive, no synchronisation)
}

}  // namespace

extern "C" int pimd_step(pimd_ctx *c, int n)
{
    if (!c || n < 0) { pimd_set_error("invalid argument"); return PIMD_ERR_ARG; }
    if (c->step + n > PIMD_MAX_STEP) { pimd_set_error("step counter would exceed 2^32 - 1 (the noise counter holds 32 bits)"); return PIMD_ERR_ARG; }
    int rc;
    if ((rc = enter(c))) return rc;
    if (!c->forces_valid && (rc = compute_forces(c))) return rc;   // (also sets every opt-in kernel attribute before a capture)
    const bool profiling = (c->prof && c->prof->on) || c->md.cv != 0;   // (metadynamics: plain launches, the deposition is decided by the host)
    // The launch sequence of a step is captured once as a CUDA graph and replayed: the small configurations are bound by
    // launch overhead (17-35 launches per step).  Per-class event timing (pimd_profile) needs the plain launches.
    for (int s = 0; s < n; ++s) {
        if (!profiling && c->graph_state == 0 && c->warm) {   // (the first step of a context runs uncaptured: lazy kernel attributes)
            c->graph_state = -1;
            cudaGraph_t g = nullptr;
            const int64_t launches0 = c->launches;
            if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
                rc = step_body(c);
                const cudaError_t e = cudaStreamEndCapture(c->stream, &g);
                c->launches_per_step = c->launches - launches0;
                c->launches = launches0;
                if (rc == 0 && e == cudaSuccess && g && cudaGraphInstantiate(&c->step_graph, g, 0) == cudaSuccess) c->graph_state = 1;
                if (g) cudaGraphDestroy(g);
            }
            (void)cudaGetLastError();
        }
        if (!profiling && c->graph_state == 1) {
            PIMD_CUDA_CHECK(cudaGraphLaunch(c->step_graph, c->stream));
            c->launches += c->launches_per_step;
            c->forces_valid = 1;
        } else {
            if ((rc = step_body(c))) return rc;
            c->warm = 1;
        }
        c->step += 1;
        if (c->md.cv && c->step % c->md.every == 0) {   // a Gaussian per bead at the positions just reached; F(q) includes them from here on
            if ((rc = pimd_launch_metad_deposit(c))) return rc;
            if ((rc = compute_forces(c))) return rc;
        }
    }
    return 0;
}

// ---- well-tempered metadynamics ---------------------------------------------------------------------
extern "C" int pimd_metad_enable(pimd_ctx *c, int cv, const int32_t *atoms6, const double *f_species, double Q, double sigma,
                                 double height_eV, double bias_factor, int deposit_every)
{
    if (!c) { pimd_set_error("null context"); return PIMD_ERR_ARG; }
    if ((cv != 1 && cv != 2) || !(sigma > 0.0) || !(bias_factor > 1.0) || deposit_every < 1 || !(height_eV >= 0.0)) {
        pimd_set_error("metadynamics: cv in {1, 2}, sigma > 0, bias factor > 1, deposit_every >= 1");
        return PIMD_ERR_ARG;
    }
    int rc;
    if ((rc = enter(c))) return rc;
    if (cv == 1) {
        if (!atoms6) { pimd_set_error("s_dimer needs six atom indices"); return PIMD_ERR_ARG; }
        for (int k = 0; k < 6; ++k) {
            if (atoms6[k] < 0 || atoms6[k] >= c->N) { pimd_set_error("s_dimer atom index %d out of range", atoms6[k]); return PIMD_ERR_ARG; }
            c->md.atoms[k] = atoms6[k];
        }
    } else {
        const int S = c->kind == 0 ? c->net.S : 16;
        if (!f_species || !(Q > 0.0) || c->N > PIMD_METAD_BLOCKS * 128) { pimd_set_error("Debye CV needs scattering factors, Q > 0 and N <= %d", PIMD_METAD_BLOCKS * 128); return PIMD_ERR_ARG; }
        for (int k = 0; k < 16; ++k) c->md.f[k] = (k < S && k < c->n_species_host) ? f_species[k] : 0.0;
        c->md.Q = Q;
    }
    c->md.sigma = sigma; c->md.w0 = height_eV; c->md.biasf = bias_factor; c->md.every = deposit_every;
    PIMD_CUDA_CHECK(cudaMemsetAsync(c->md.n_g, 0, sizeof(int) * (size_t)c->R, c->stream));
    PIMD_CUDA_CHECK(cudaMemsetAsync(c->md.grad, 0, sizeof(double) * (size_t)c->rows * 3, c->stream));
    c->md.cv = cv;
    c->forces_valid = 0;
    drop_step_graph(c);
    return 0;
}

extern "C" int pimd_metad_cv(pimd_ctx *c, double *d_s, double *d_grad)
{
    if (!c || !c->md.cv) { pimd_set_error("metadynamics is not enabled"); return PIMD_ERR_ARG; }
    int rc;
    if ((rc = enter(c))) return rc;
    if ((rc = pimd_launch_metad_bias(c, 0))) return rc;
    if (d_s) PIMD_CUDA_CHECK(cudaMemcpyAsync(d_s, c->md.s, sizeof(double) * (size_t)c->R * c->P, cudaMemcpyDeviceToDevice, c->stream));
    if (d_grad) PIMD_CUDA_CHECK(cudaMemcpyAsync(d_grad, c->md.grad, sizeof(double) * (size_t)c->rows * 3, cudaMemcpyDeviceToDevice, c->stream));
    return 0;
}

extern "C" int pimd_metad_gaussians(pimd_ctx *c, int replica, double *h_centres, double *h_heights, int cap, int *h_n)
{
    if (!c || !c->md.cv || !h_n || replica < 0 || replica >= c->R) { pimd_set_error("invalid argument"); return PIMD_ERR_ARG; }
    int rc;
    if ((rc = enter(c))) return rc;
    int n = 0;
    PIMD_CUDA_CHECK(cudaMemcpyAsync(&n, c->md.n_g + replica, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    PIMD_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    *h_n = n;
    const int m = n < cap ? n : cap;
    if (m > 0 && h_centres) PIMD_CUDA_CHECK(cudaMemcpyAsync(h_centres, c->md.gc + (size_t)replica * PIMD_METAD_MAX, sizeof(double) * m, cudaMemcpyDeviceToHost, c->stream));
    if (m > 0 && h_heights) PIMD_CUDA_CHECK(cudaMemcpyAsync(h_heights, c->md.gh + (size_t)replica * PIMD_METAD_MAX, sizeof(double) * m, cudaMemcpyDeviceToHost, c->stream));
    PIMD_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    return 0;
}

extern "C" int pimd_metad_deposit_now(pimd_ctx *c)
{
    if (!c || !c->md.cv) { pimd_set_error("metadynamics is not enabled"); return PIMD_ERR_ARG; }
    int rc;
    if ((rc = enter(c))) return rc;
    if (!c->forces_valid && (rc = compute_forces(c))) return rc;   // the CV values of the current positions
    if ((rc = pimd_launch_metad_deposit(c))) return rc;
    c->forces_valid = 0;
    return 0;
}

extern "C" int pimd_forces(pimd_ctx *c, float *d_out)
{
    if (!c || !d_out) { pimd_set_error("null argument"); return PIMD_ERR_ARG; }
    int rc;
    if ((rc = enter(c))) return rc;
    if ((rc = compute_forces(c))) return rc;
    return pimd_launch_copy_forces_f32(c, d_out);
}

extern "C" int pimd_estimators(pimd_ctx *c, pimd_estimators_t *h_out)
{
    if (!c || !h_out) { pimd_set_error("null argument"); return PIMD_ERR_ARG; }
    int rc;
    if ((rc = enter(c))) return rc;
    if (!c->forces_valid && (rc = compute_forces(c))) return rc;
    if ((rc = pimd_launch_estimators(c))) return rc;
    std::vector<double> tmp((size_t)c->R * 8);
    PIMD_CUDA_CHECK(cudaMemcpyAsync(tmp.data(), c->est_out, sizeof(double) * tmp.size(), cudaMemcpyDeviceToHost, c->stream));
    if ((rc = check_device_error(c))) return rc;   // synchronises
    for (int r = 0; r < c->R; ++r) {
        h_out[r].k_prim = tmp[r * 8 + 0]; h_out[r].k_vir = tmp[r * 8 + 1]; h_out[r].k_cvir = tmp[r * 8 + 2];
        h_out[r].v_pot = tmp[r * 8 + 3]; h_out[r].t_centroid = tmp[r * 8 + 4];
    }
    return 0;
}

extern "C" int pimd_get_state(pimd_ctx *c, double *d_q, double *d_p, int64_t *step)
{
    if (!c) { pimd_set_error("null context"); return PIMD_ERR_ARG; }
    if (int rc = enter(c)) return rc;
    const size_t bytes = sizeof(double) * (size_t)c->rows * 3;
    if (d_q) PIMD_CUDA_CHECK(cudaMemcpyAsync(d_q, c->q, bytes, cudaMemcpyDefault, c->stream));
    if (d_p) PIMD_CUDA_CHECK(cudaMemcpyAsync(d_p, c->p, bytes, cudaMemcpyDefault, c->stream));
    if (step) *step = c->step;
    return check_device_error(c);
}

extern "C" int pimd_set_state(pimd_ctx *c, const double *d_q, const double *d_p, int64_t step)
{
    if (!c) { pimd_set_error("null context"); return PIMD_ERR_ARG; }
    if (step < 0 || step > PIMD_MAX_STEP) { pimd_set_error("step %lld outside [0, 2^32 - 1] (the noise counter holds 32 bits)", (long long)step); return PIMD_ERR_ARG; }
    if (int rc = enter(c)) return rc;
    const size_t bytes = sizeof(double) * (size_t)c->rows * 3;
    if (d_q) PIMD_CUDA_CHECK(cudaMemcpyAsync(c->q, d_q, bytes, cudaMemcpyDefault, c->stream));
    if (d_p) PIMD_CUDA_CHECK(cudaMemcpyAsync(c->p, d_p, bytes, cudaMemcpyDefault, c->stream));
    c->step = step;
    c->forces_valid = 0;
    if (int rc = sync_step_counter(c)) return rc;
    if (d_q) return pimd_launch_nlist_invalidate(c);   // positions jumped: the candidate lists are rebuilt at the next force evaluation
    return 0;
}

extern "C" int pimd_nlist_rebuilds(pimd_ctx *c, int64_t *h_count)
{
    if (!c || !h_count) { pimd_set_error("null argument"); return PIMD_ERR_ARG; }
    if (int rc = enter(c)) return rc;
    int v = 0;
    if (c->kind == 0) PIMD_CUDA_CHECK(cudaMemcpyAsync(&v, c->nl.need + 1, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    PIMD_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    *h_count = v;
    return 0;
}

extern "C" int pimd_set_nlist_skin(pimd_ctx *c, double skin)
{
    if (!c) { pimd_set_error("null context"); return PIMD_ERR_ARG; }
    if (int rc = enter(c)) return rc;
    return apply_skin(c, skin);
}

extern "C" int pimd_get_forces_cached(pimd_ctx *c, double *d_F)
{
    if (!c || !d_F) { pimd_set_error("null argument"); return PIMD_ERR_ARG; }
    int rc;
    if ((rc = enter(c))) return rc;
    if (!c->forces_valid && (rc = compute_forces(c))) return rc;
    PIMD_CUDA_CHECK(cudaMemcpyAsync(d_F, c->F, sizeof(double) * (size_t)c->rows * 3, cudaMemcpyDefault, c->stream));
    return 0;
}

extern "C" int pimd_set_forces_cached(pimd_ctx *c, const double *d_F)
{
    if (!c || !d_F) { pimd_set_error("null argument"); return PIMD_ERR_ARG; }
    if (int rc = enter(c)) return rc;
    PIMD_CUDA_CHECK(cudaMemcpyAsync(c->F, d_F, sizeof(double) * (size_t)c->rows * 3, cudaMemcpyDefault, c->stream));
    c->forces_valid = 1;
    return 0;
}

extern "C" int pimd_nlist(pimd_ctx *c, int32_t *d_row_ptr, int32_t *d_col, int64_t col_capacity, int64_t *h_n_pairs)
{
    if (!c || !d_row_ptr || !d_col || !h_n_pairs) { pimd_set_error("null argument"); return PIMD_ERR_ARG; }
    if (c->kind != 0) { pimd_set_error("no neighbour list for this potential kind"); return PIMD_ERR_ARG; }
    int rc;
    if ((rc = enter(c))) return rc;
    if ((rc = pimd_launch_nlist(c))) return rc;
    int n = 0;
    PIMD_CUDA_CHECK(cudaMemcpyAsync(&n, c->nl.row_ptr + c->rows, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    if ((rc = check_device_error(c))) return rc;
    *h_n_pairs = n;
    if (n > col_capacity) { pimd_set_error("col_capacity %lld < %d pairs", (long long)col_capacity, n); return PIMD_ERR_PAIRS; }
    PIMD_CUDA_CHECK(cudaMemcpyAsync(d_row_ptr, c->nl.row_ptr, sizeof(int) * (c->rows + 1), cudaMemcpyDeviceToDevice, c->stream));
    PIMD_CUDA_CHECK(cudaMemcpyAsync(d_col, c->nl.col, sizeof(int) * (size_t)n, cudaMemcpyDeviceToDevice, c->stream));
    PIMD_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    return 0;
}

extern "C" int pimd_sync(pimd_ctx *c)
{
    if (!c) { pimd_set_error("null context"); return PIMD_ERR_ARG; }
    if (int rc = enter(c)) return rc;
    return check_device_error(c);
}

extern "C" int pimd_profile(pimd_ctx *c, int enable)
{
    if (!c) { pimd_set_error("null context"); return PIMD_ERR_ARG; }
    if (!c->prof) c->prof = new PimdProf();
    PIMD_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    if (enable) c->prof->clear();
    c->prof->on = enable != 0;
    return 0;
}

extern "C" int pimd_profile_read(pimd_ctx *c, double *h_ms, int64_t *h_launches)
{
    if (!c || !h_ms || !h_launches) { pimd_set_error("null argument"); return PIMD_ERR_ARG; }
    for (int k = 0; k < PIMD_PROF_CLASSES; ++k) { h_ms[k] = 0.0; h_launches[k] = 0; }
    if (!c->prof) return 0;
    PIMD_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    for (auto &r : c->prof->recs) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, r.a, r.b) != cudaSuccess) { (void)cudaGetLastError(); continue; }
        h_ms[r.kind] += ms;
        h_launches[r.kind] += 1;
    }
    return 0;
}

extern "C" int64_t pimd_launch_count(const pimd_ctx *c) { return c ? c->launches : 0; }
