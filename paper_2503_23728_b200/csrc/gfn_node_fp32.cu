// gfn_node_fp32.cu -- atom-wise dense layers of the GFN force net, fp32 FFMA version
// (rows a4 and a6 of SURVEY 8(a); P:L74 phi_v and the node->edge MLP of P:L76), the force
// finalisation, and the host-side sequencing of one force evaluation.
//
// One CTA owns a 128-row tile and runs the whole node update on it with the activations resident in
// shared memory (k-major, swizzled) and the H x H weight matrices streamed through a 64 KB slab:
//   h   = SiLU(W_vn n + W_vm m + b_v1)          m assembled from direct rows + carry slots
//   n  += W_v2 h + b_v2
//   E  += W_a n + b_a                            (running sum of the edge updates, S:G5)
//   x   = W_s^{l+1} n      or, after the last layer,   G = W_f1 E
#include "gfn_fp32.cuh"

namespace gfn {

int launch_pair(pimd_ctx *c, int layer, bool head);

struct NodeArgs {
    int N, mode;                 // mode 0: INIT (n = Emb[species], E = 0, x = W_s0 n); 1: layer update
    int last;                    // layer update: 1 -> write G = W_f1 E instead of x
    int64_t rows;
    const int *species, *row_ptr;
    int gran_m;
    const float *Emb;
    const float *WvnT, *WvmT, *bv1, *Wv2T, *bv2, *WaT, *ba, *WnextT;
    float *n, *E, *out;          // out = x or G
    const float *m, *carry_m;
};

template <int H>
struct NodeSmem {
    float W[H * H];
    float A[H * TP];
    float B[H * TP];
    float bv1[H], bv2[H], ba[H];
};

// m_i assembled in fixed order: direct row, or tail slot of the first granule + head slots of the rest
__device__ __forceinline__ float4 assemble_m(const NodeArgs &a, int64_t row, int c0, int H, int n_pairs)
{
    const int rs = a.row_ptr[row], re = a.row_ptr[row + 1];
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (re <= rs || n_pairs == 0) return v;
    const int g0 = rs / a.gran_m, g1 = (re - 1) / a.gran_m;
    if (g0 == g1) return __ldg((const float4 *)(a.m + (size_t)row * H + c0));
    v = __ldg((const float4 *)(a.carry_m + ((size_t)g0 * 2 + 1) * H + c0));
    for (int g = g0 + 1; g <= g1; ++g) {
        float4 t = __ldg((const float4 *)(a.carry_m + ((size_t)g * 2 + 0) * H + c0));
        v.x += t.x; v.y += t.y; v.z += t.z; v.w += t.w;
    }
    return v;
}

// RP = 8: 128-row tiles; RP = 4 / 2: 64- / 32-row tiles (the first rows of the same buffers) when there are fewer tiles than SMs
template <int H, int RP>
__global__ void __launch_bounds__(NT, 1) node_kernel(NodeArgs a)
{ pdl_enter();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    NodeSmem<H> &S = *reinterpret_cast<NodeSmem<H> *>(smem_raw);
    constexpr int CPT = Tile<H>::CPT;
    const int tid = threadIdx.x, tx = tid % TX, ty = tid / TX;
    constexpr int TPv = 16 * RP;                   // rows of this CTA's tile
    const int64_t row0 = (int64_t)blockIdx.x * TPv;
    const int n_pairs = a.row_ptr[a.rows];

    // The weight matrices go through one shared-memory slab, each load in front of its product.  A layer's matrices are touched
    // once per step: their lines are requested into L2 now, so that the five loads below do not each pay a DRAM round trip.
    {
        const float *mats[5] = {a.mode == 1 ? a.WvnT : nullptr, a.mode == 1 ? a.WvmT : nullptr, a.mode == 1 ? a.Wv2T : nullptr,
                                a.mode == 1 ? a.WaT : nullptr, a.WnextT};
#pragma unroll
        for (int m = 0; m < 5; ++m)
            if (mats[m])
                for (int i = tid * 32; i < H * H; i += NT * 32) asm volatile("prefetch.global.L2 [%0];" ::"l"(mats[m] + i));
    }

    // ---- load the tile transposed into the k-major buffers
    for (int idx = tid; idx < TPv * H / 4; idx += NT) {
        const int r = idx / (H / 4), c4 = idx % (H / 4), c0 = c4 * 4;
        const int64_t row = row0 + r;
        float4 nv = make_float4(0.f, 0.f, 0.f, 0.f), mv = nv;
        if (row < a.rows) {
            if (a.mode == 0) {
                nv = __ldg((const float4 *)(a.Emb + (size_t)a.species[row % a.N] * H + c0));
                *(float4 *)(a.n + (size_t)row * H + c0) = nv;
                *(float4 *)(a.E + (size_t)row * H + c0) = make_float4(0.f, 0.f, 0.f, 0.f);
            } else {
                nv = *(const float4 *)(a.n + (size_t)row * H + c0);
                mv = assemble_m(a, row, c0, H, n_pairs);
            }
        }
        const int col = r ^ swz(c0);
        S.A[(c0 + 0) * TP + col] = nv.x; S.A[(c0 + 1) * TP + col] = nv.y;
        S.A[(c0 + 2) * TP + col] = nv.z; S.A[(c0 + 3) * TP + col] = nv.w;
        if (a.mode == 1) {
            S.B[(c0 + 0) * TP + col] = mv.x; S.B[(c0 + 1) * TP + col] = mv.y;
            S.B[(c0 + 2) * TP + col] = mv.z; S.B[(c0 + 3) * TP + col] = mv.w;
        }
    }
    float acc[RP][CPT];

    if (a.mode == 1) {
        for (int i = tid; i < H; i += NT) { S.bv1[i] = a.bv1[i]; S.bv2[i] = a.bv2[i]; S.ba[i] = a.ba[i]; }
        load_matrix<H>(S.W, a.WvnT, H);
        __syncthreads();
        zero_acc<H, RP>(acc);
        tile_gemm<H, H, RP>(S.A, S.W, acc, tx, ty);          // W_vn n
        __syncthreads();
        load_matrix<H>(S.W, a.WvmT, H);
        __syncthreads();
        tile_gemm<H, H, RP>(S.B, S.W, acc, tx, ty);          // + W_vm m
        __syncthreads();
#pragma unroll
        for (int c = 0; c < CPT; ++c) {
            const float b = S.bv1[Tile<H>::chan(tx, c >> 2, c & 3)];
#pragma unroll
            for (int p = 0; p < RP; ++p) acc[p][c] = silu_f(acc[p][c] + b);
        }
        store_as_A<H, RP>(S.B, acc, tx, ty);                 // h
        load_matrix<H>(S.W, a.Wv2T, H);
        __syncthreads();
        zero_acc<H, RP>(acc);
        tile_gemm<H, H, RP>(S.B, S.W, acc, tx, ty);          // W_v2 h
        // n <- n + W_v2 h + b_v2   (this thread's own elements of A; A is not read by the GEMM above)
#pragma unroll
        for (int c = 0; c < CPT; ++c) {
            const int ch = Tile<H>::chan(tx, c >> 2, c & 3);
            const float b = S.bv2[ch];
#pragma unroll
            for (int p = 0; p < RP; ++p) {
                const int pr = tile_row<RP>(ty, p);
                acc[p][c] += S.A[ch * TP + (pr ^ swz(ch))] + b;
            }
        }
        __syncthreads();
        store_as_A<H, RP>(S.A, acc, tx, ty);                 // updated n
#pragma unroll
        for (int p = 0; p < RP; ++p) {
            const int64_t row = row0 + tile_row<RP>(ty, p);
            if (row < a.rows)
#pragma unroll
                for (int g = 0; g < CPT / 4; ++g)
                    *(float4 *)(a.n + (size_t)row * H + Tile<H>::chan(tx, g, 0)) =
                        make_float4(acc[p][g * 4], acc[p][g * 4 + 1], acc[p][g * 4 + 2], acc[p][g * 4 + 3]);
        }
        load_matrix<H>(S.W, a.WaT, H);
        __syncthreads();
        zero_acc<H, RP>(acc);
        tile_gemm<H, H, RP>(S.A, S.W, acc, tx, ty);          // a = W_a n + b_a ; E += a
#pragma unroll
        for (int p = 0; p < RP; ++p) {
            const int64_t row = row0 + tile_row<RP>(ty, p);
#pragma unroll
            for (int g = 0; g < CPT / 4; ++g) {
                const int c0 = Tile<H>::chan(tx, g, 0);
                float4 e = make_float4(0.f, 0.f, 0.f, 0.f);
                if (row < a.rows) e = *(const float4 *)(a.E + (size_t)row * H + c0);
                acc[p][g * 4 + 0] += e.x + S.ba[c0 + 0]; acc[p][g * 4 + 1] += e.y + S.ba[c0 + 1];
                acc[p][g * 4 + 2] += e.z + S.ba[c0 + 2]; acc[p][g * 4 + 3] += e.w + S.ba[c0 + 3];
                if (row < a.rows)
                    *(float4 *)(a.E + (size_t)row * H + c0) =
                        make_float4(acc[p][g * 4], acc[p][g * 4 + 1], acc[p][g * 4 + 2], acc[p][g * 4 + 3]);
            }
        }
        if (a.last) store_as_A<H, RP>(S.B, acc, tx, ty);     // E as the operand of G = W_f1 E
        __syncthreads();
    }
    // ---- x = W_s n   (or G = W_f1 E)
    load_matrix<H>(S.W, a.WnextT, H);
    __syncthreads();
    zero_acc<H, RP>(acc);
    tile_gemm<H, H, RP>((a.mode == 1 && a.last) ? S.B : S.A, S.W, acc, tx, ty);
#pragma unroll
    for (int p = 0; p < RP; ++p) {
        const int64_t row = row0 + tile_row<RP>(ty, p);
        if (row < a.rows)
#pragma unroll
            for (int g = 0; g < CPT / 4; ++g)
                *(float4 *)(a.out + (size_t)row * H + Tile<H>::chan(tx, g, 0)) =
                    make_float4(acc[p][g * 4], acc[p][g * 4 + 1], acc[p][g * 4 + 2], acc[p][g * 4 + 3]);
    }
}

// F_i = force_scale * (direct row sum, or carry slots in fixed order) -> fp64 force array
__global__ void force_finalize_kernel(int64_t rows, const int *__restrict__ row_ptr, int gran, float force_scale,
                                      const float *__restrict__ Fraw, const float *__restrict__ carry,
                                      double *__restrict__ F)
{ pdl_enter();
    int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= rows) return;
    const int rs = row_ptr[row], re = row_ptr[row + 1];
    float v[3] = {0.f, 0.f, 0.f};
    if (re > rs && row_ptr[rows] > 0) {
        const int g0 = rs / gran, g1 = (re - 1) / gran;
        if (g0 == g1) {
            for (int ax = 0; ax < 3; ++ax) v[ax] = Fraw[row * 4 + ax];
        } else {
            for (int ax = 0; ax < 3; ++ax) v[ax] = carry[((size_t)g0 * 2 + 1) * 4 + ax];
            for (int g = g0 + 1; g <= g1; ++g)
                for (int ax = 0; ax < 3; ++ax) v[ax] += carry[((size_t)g * 2 + 0) * 4 + ax];
        }
    }
    for (int ax = 0; ax < 3; ++ax) F[row * 3 + ax] = (double)(force_scale * v[ax]);
}

template <int H>
int launch_node_t(pimd_ctx *c, const NodeArgs &a)
{
    size_t smem = sizeof(NodeSmem<H>);
    if (!(c->attr_done & ATTR_NODE32)) {
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(node_kernel<H, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(node_kernel<H, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(node_kernel<H, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        c->attr_done |= ATTR_NODE32;
    }
    if (c->rows <= (int64_t)(TP / 4) * c->num_sms) // quarter tiles still fit one per SM
        pimd_launch(node_kernel<H, 2>, (unsigned)((c->rows + TP / 4 - 1) / (TP / 4)), NT, smem, c->stream, a);
    else if (c->rows < (int64_t)TP * c->num_sms)   // fewer 128-row tiles than SMs: half tiles, twice the CTAs
        pimd_launch(node_kernel<H, 4>, (unsigned)((c->rows + TP / 2 - 1) / (TP / 2)), NT, smem, c->stream, a);
    else
        pimd_launch(node_kernel<H, 8>, (unsigned)((c->rows + TP - 1) / TP), NT, smem, c->stream, a);
    c->launches++;
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}

}  // namespace gfn
namespace node_tc { int launch_node_tc(pimd_ctx *c, int mode, int layer); }
namespace gfn {

int launch_node(pimd_ctx *c, int mode, int layer)
{
    if (c->use_tc) return node_tc::launch_node_tc(c, mode, layer);
    const GfnDev &n = c->net;
    NodeArgs a;
    a.N = c->N; a.mode = mode; a.rows = c->rows; a.species = c->species; a.row_ptr = c->nl.row_ptr;
    a.gran_m = c->gran_m; a.Emb = n.Emb;
    a.n = c->nfeat; a.E = c->Efeat; a.m = c->mfeat; a.carry_m = c->carry_m;
    if (mode == 0) {
        a.last = 0;
        a.WvnT = a.WvmT = a.bv1 = a.Wv2T = a.bv2 = a.WaT = a.ba = nullptr;
        a.WnextT = n.layer[0].WsT; a.out = c->xfeat;
    } else {
        const GfnLayerW &w = n.layer[layer];
        a.last = (layer == n.L - 1);
        a.WvnT = w.WvnT; a.WvmT = w.WvmT; a.bv1 = w.bv1; a.Wv2T = w.Wv2T; a.bv2 = w.bv2; a.WaT = w.WaT; a.ba = w.ba;
        a.WnextT = a.last ? n.Wf1T : n.layer[layer + 1].WsT;
        a.out = a.last ? c->Gfeat : c->xfeat;
    }
    if (n.H == 64) return launch_node_t<64>(c, a);
    if (n.H == 128) return launch_node_t<128>(c, a);
    pimd_set_error("unsupported hidden = %d", n.H);
    return PIMD_ERR_ARG;
}

}  // namespace gfn

bool pimd_gfn_supported(int K, int H) { return (K == 32 && H == 64) || (K == 64 && H == 128); }

// One force evaluation on the current neighbour list (S:G3, G4)
int pimd_launch_gfn_forces(pimd_ctx *c)
{
    int rc;
    const int L = c->net.L;
    if (L == 0) {
        PIMD_CUDA_CHECK(cudaMemsetAsync(c->Gfeat, 0, sizeof(float) * (size_t)c->rows * c->net.H, c->stream));
    } else {
        {
            ProfScope ps(c, PROF_NODE);
            if ((rc = gfn::launch_node(c, 0, 0))) return rc;
        }
        for (int l = 0; l < L; ++l) {
            {
                ProfScope ps(c, PROF_PAIR);
                if ((rc = gfn::launch_pair(c, l, false))) return rc;
            }
            ProfScope ps(c, PROF_NODE);
            if ((rc = gfn::launch_node(c, 1, l))) return rc;
        }
    }
    {
        ProfScope ps(c, PROF_HEAD);
        if ((rc = gfn::launch_pair(c, L, true))) return rc;
    }
    ProfScope ps(c, PROF_OTHER);
    pimd_launch(gfn::force_finalize_kernel, (unsigned)((c->rows + 255) / 256), 256, 0, c->stream, 
        c->rows, c->nl.row_ptr, c->gran_f, c->net.force_scale, c->Fraw, c->carry_f, c->F);
    c->launches++;
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}
