// gfn_pair_fp32.cu -- fused per-pair kernels of the GFN force net, fp32 FFMA version
// (rows a5 and a7 of SURVEY 8(a); P:L74 phi_m / agg, P:L76 edge MLP, P:L78 force readout).
//
// One persistent CTA per SM walks 128-pair tiles of the flat CSR pair list.  Per tile:
//   geometry in fp64 (minimum image) -> Gaussian RBF tile in shared memory -> filter MLP as two
//   register-tiled GEMMs against weights resident in shared memory (SiLU between them) ->
//   epilogue with the running-sum edge state e_ij = e0_ij + E_i + E_j (S:G5):
//     MESSAGE: val = agg_norm c_ij e_ij (.) x_j, deterministic segmented sum over the CSR rows
//     HEAD:    s_ij = w_f2 . SiLU((W_f1 W_e2) h1 + W_f1 b_e2 + b_f1 + G_i + G_j) + b_f2 with G = W_f1 E
//              (W_f1 is linear, so W_f1 e_ij splits exactly), F_i = sum_j c_ij s_ij u_ij by a
//              segmented warp reduction.
// Rows that straddle a reduction granule go through carry slots that the consumer adds in a fixed
// order: no floating-point atomics anywhere.
#include "gfn_fp32.cuh"

namespace gfn {

struct PairArgs {
    int N, periodic;
    double box[3];
    float r_cut, wscale;          // wscale: agg_norm (message) or 1 (head)
    const int *row_ptr, *col, *pair_row;
    int64_t rows;
    const double *q;
    const float *W1T, *b1, *W2T, *b2;     // filter MLP (W2 = W_e2 or W_f1 W_e2)
    const float *Ea, *xa;                 // message: E, x ; head: G, unused
    const float *wf2; float bf2;
    float *m_out, *carry_m;               // message outputs
    float *Fraw, *carry_f;                // head outputs
};

template <int K, int H>
struct PairSmem {
    static constexpr int KA = (K > H ? K : H);
    float W1[K * H];
    float W2[H * H];
    float A[KA * TP];
    float b1[H], b2[H], wf2[H];
    double d[TP];
    float w[TP], u[TP][3], s[TP];
    int row[TP], jrow[TP], rs[TP], re[TP];
};

template <int K, int H, bool HEAD>
__global__ void __launch_bounds__(NT, 1) pair_kernel(PairArgs a)
{ pdl_enter();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    PairSmem<K, H> &S = *reinterpret_cast<PairSmem<K, H> *>(smem_raw);
    constexpr int CPT = Tile<H>::CPT;
    const int tid = threadIdx.x, tx = tid % TX, ty = tid / TX;
    const int64_t n_pairs = a.row_ptr[a.rows];
    if ((int64_t)blockIdx.x * TP >= n_pairs) return;

    load_matrix<H>(S.W1, a.W1T, K);
    load_matrix<H>(S.W2, a.W2T, H);
    for (int i = tid; i < H; i += NT) {
        S.b1[i] = a.b1[i]; S.b2[i] = a.b2[i];
        S.wf2[i] = HEAD ? a.wf2[i] : 0.f;
    }
    const double delta = (double)a.r_cut / (K - 1), inv_delta = 1.0 / delta;

    for (int64_t tile0 = (int64_t)blockIdx.x * TP; tile0 < n_pairs; tile0 += (int64_t)gridDim.x * TP) {
        __syncthreads();   // previous tile fully consumed; weights visible
        // ---- per-pair geometry (S:G1), fp64 minimum image
        if (tid < TP) {
            int64_t p = tile0 + tid;
            int row = -1, jrow = 0, rs = 0, re = 0;
            double dist = 0.0;
            float w = 0.f, ux = 0.f, uy = 0.f, uz = 0.f;
            if (p < n_pairs) {
                row = a.pair_row[p];
                int sys = row / a.N;
                jrow = sys * a.N + a.col[p];
                rs = a.row_ptr[row]; re = a.row_ptr[row + 1];
                double dv[3];
#pragma unroll
                for (int ax = 0; ax < 3; ++ax) {
                    double dx = a.q[(size_t)jrow * 3 + ax] - a.q[(size_t)row * 3 + ax];
                    if (a.periodic) dx = dx - a.box[ax] * round(dx / a.box[ax]);
                    dv[ax] = dx;
                }
                dist = sqrt(dv[0] * dv[0] + dv[1] * dv[1] + dv[2] * dv[2]);
                double inv = 1.0 / fmax(dist, 1e-12);
                ux = (float)(-dv[0] * inv); uy = (float)(-dv[1] * inv); uz = (float)(-dv[2] * inv);
                w = a.wscale * 0.5f * (cospif((float)(dist / (double)a.r_cut)) + 1.0f);
            }
            S.row[tid] = row; S.jrow[tid] = jrow; S.rs[tid] = rs; S.re[tid] = re;
            S.d[tid] = dist; S.w[tid] = w; S.u[tid][0] = ux; S.u[tid][1] = uy; S.u[tid][2] = uz;
        }
        __syncthreads();
        // ---- Gaussian RBF tile g_k(d) = exp(-(d - k delta)^2 / (2 delta^2)) -> A[k][p]
        for (int idx = tid; idx < K * TP; idx += NT) {
            int k = idx / TP, p = idx % TP;
            float t = (float)((S.d[p] - k * delta) * inv_delta);
            S.A[k * TP + (p ^ swz(k))] = __expf(-0.5f * t * t);
        }
        __syncthreads();
        // ---- h1 = SiLU(W_e1 g + b_e1)
        float acc[8][CPT];
        zero_acc<H>(acc);
        tile_gemm<K, H>(S.A, S.W1, acc, tx, ty);
        __syncthreads();
#pragma unroll
        for (int c = 0; c < CPT; ++c) {
            float b = S.b1[Tile<H>::chan(tx, c >> 2, c & 3)];
#pragma unroll
            for (int p = 0; p < 8; ++p) acc[p][c] = silu_f(acc[p][c] + b);
        }
        store_as_A<H>(S.A, acc, tx, ty);
        __syncthreads();
        // ---- second filter layer (W_e2, or W_f1 W_e2 for the head)
        zero_acc<H>(acc);
        tile_gemm<H, H>(S.A, S.W2, acc, tx, ty);
        __syncthreads();   // everybody is done reading A; it is reused below as the message tile

        if (!HEAD) {
            // val[p][c] = w_p (e0 + E_i + E_j)[c] x_j[c]  -> msg[p][c] (row-major [TP][H])
            float *msg = S.A;
#pragma unroll
            for (int pi = 0; pi < 8; ++pi) {
                const int p = Tile<H>::pair(ty, pi >> 2, pi & 3);
                const int row = S.row[p], jrow = S.jrow[p];
                const float w = S.w[p];
#pragma unroll
                for (int g = 0; g < CPT / 4; ++g) {
                    const int c0 = Tile<H>::chan(tx, g, 0);
                    float4 out = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (row >= 0) {
                        float4 Ei = __ldg((const float4 *)(a.Ea + (size_t)row * H + c0));
                        float4 Ej = __ldg((const float4 *)(a.Ea + (size_t)jrow * H + c0));
                        float4 xj = __ldg((const float4 *)(a.xa + (size_t)jrow * H + c0));
                        out.x = w * (acc[pi][g * 4 + 0] + S.b2[c0 + 0] + Ei.x + Ej.x) * xj.x;
                        out.y = w * (acc[pi][g * 4 + 1] + S.b2[c0 + 1] + Ei.y + Ej.y) * xj.y;
                        out.z = w * (acc[pi][g * 4 + 2] + S.b2[c0 + 2] + Ei.z + Ej.z) * xj.z;
                        out.w = w * (acc[pi][g * 4 + 3] + S.b2[c0 + 3] + Ei.w + Ej.w) * xj.w;
                    }
                    *(float4 *)&msg[p * H + c0] = out;
                }
            }
            __syncthreads();
            // deterministic segmented sum: thread (part, ch) walks its granule of pairs in CSR order
            constexpr int NPART = NT / H, GP = TP / NPART;
            const int ch = tid % H, part = tid / H;
            const int64_t g0 = tile0 + (int64_t)part * GP, g1 = g0 + GP;
            const int64_t gidx = g0 / GP;
            int cur = -1, pfirst = 0;
            float sum = 0.f;
            for (int pp = 0; pp <= GP; ++pp) {
                const int p = part * GP + pp;
                const int r = (pp < GP) ? S.row[p] : -2;
                if (r != cur) {
                    if (cur >= 0) {
                        const int rs = S.rs[pfirst], re = S.re[pfirst];
                        if (rs >= g0 && re <= g1) a.m_out[(size_t)cur * H + ch] = sum;
                        else if (rs < g0) a.carry_m[(size_t)(gidx * 2 + 0) * H + ch] = sum;
                        else a.carry_m[(size_t)(gidx * 2 + 1) * H + ch] = sum;
                    }
                    cur = r; pfirst = p; sum = 0.f;
                }
                if (r >= 0) sum += msg[p * H + ch];
            }
        } else {
            // s_p = w_f2 . SiLU(acc + b_fe + G_i + G_j) + b_f2
            float part[8];
#pragma unroll
            for (int pi = 0; pi < 8; ++pi) {
                const int p = Tile<H>::pair(ty, pi >> 2, pi & 3);
                const int row = S.row[p], jrow = S.jrow[p];
                float s = 0.f;
                if (row >= 0) {
#pragma unroll
                    for (int g = 0; g < CPT / 4; ++g) {
                        const int c0 = Tile<H>::chan(tx, g, 0);
                        float4 Gi = __ldg((const float4 *)(a.Ea + (size_t)row * H + c0));
                        float4 Gj = __ldg((const float4 *)(a.Ea + (size_t)jrow * H + c0));
                        s += S.wf2[c0 + 0] * silu_f(acc[pi][g * 4 + 0] + S.b2[c0 + 0] + Gi.x + Gj.x);
                        s += S.wf2[c0 + 1] * silu_f(acc[pi][g * 4 + 1] + S.b2[c0 + 1] + Gi.y + Gj.y);
                        s += S.wf2[c0 + 2] * silu_f(acc[pi][g * 4 + 2] + S.b2[c0 + 2] + Gi.z + Gj.z);
                        s += S.wf2[c0 + 3] * silu_f(acc[pi][g * 4 + 3] + S.b2[c0 + 3] + Gi.w + Gj.w);
                    }
                }
                part[pi] = s;
            }
#pragma unroll
            for (int pi = 0; pi < 8; ++pi) {   // sum over the 16 channel groups (a half-warp), fixed tree
#pragma unroll
                for (int o = 8; o > 0; o >>= 1) part[pi] += __shfl_xor_sync(0xffffffffu, part[pi], o);
                if (tx == 0) S.s[Tile<H>::pair(ty, pi >> 2, pi & 3)] = part[pi] + a.bf2;
            }
            __syncthreads();
            // segmented warp reduction over 32-pair granules (rows are contiguous in the CSR)
            if (tid < TP) {
                const int lane = tid & 31;
                const int key = S.row[tid];
                const float f = S.w[tid] * S.s[tid];
                float v[3] = {f * S.u[tid][0], f * S.u[tid][1], f * S.u[tid][2]};
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    int ko = __shfl_up_sync(0xffffffffu, key, o);
#pragma unroll
                    for (int ax = 0; ax < 3; ++ax) {
                        float vo = __shfl_up_sync(0xffffffffu, v[ax], o);
                        if (lane >= o && ko == key) v[ax] += vo;
                    }
                }
                int knext = __shfl_down_sync(0xffffffffu, key, 1);
                if (key >= 0 && (lane == 31 || knext != key)) {
                    const int64_t g0 = tile0 + (tid & ~31), g1 = g0 + 32, gidx = g0 >> 5;
                    const int rs = S.rs[tid], re = S.re[tid];
                    float *dst;
                    if (rs >= g0 && re <= g1) dst = a.Fraw + (size_t)key * 4;
                    else if (rs < g0) dst = a.carry_f + (size_t)(gidx * 2 + 0) * 4;
                    else dst = a.carry_f + (size_t)(gidx * 2 + 1) * 4;
                    dst[0] = v[0]; dst[1] = v[1]; dst[2] = v[2];
                }
            }
        }
    }
}

template <int K, int H>
int launch_pair_t(pimd_ctx *c, const PairArgs &a, bool head)
{
    size_t smem = sizeof(PairSmem<K, H>);
    if (!(c->attr_done & ATTR_PAIR32)) {
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(pair_kernel<K, H, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(pair_kernel<K, H, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        c->attr_done |= ATTR_PAIR32;
    }
    if (head) pimd_launch(pair_kernel<K, H, true>, c->num_sms, NT, smem, c->stream, a);
    else pimd_launch(pair_kernel<K, H, false>, c->num_sms, NT, smem, c->stream, a);
    c->launches++;
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}

}  // namespace gfn
namespace gfn_pipe { int launch_pair_pipe(pimd_ctx *c, bool head, bool first); }
namespace gfn {

int launch_pair(pimd_ctx *c, int layer, bool head)
{
    if (c->use_tc) return gfn_pipe::launch_pair_pipe(c, head, layer == 0);   // layer 0 = first pair pass of this evaluation
    PairArgs a;
    a.N = c->N; a.periodic = c->periodic;
    for (int k = 0; k < 3; ++k) a.box[k] = c->box[k];
    a.r_cut = c->net.r_cut; a.wscale = head ? 1.0f : c->net.agg_norm;
    a.row_ptr = c->nl.row_ptr; a.col = c->nl.col; a.pair_row = c->nl.pair_row; a.rows = c->rows; a.q = c->q;
    a.W1T = c->net.We1T; a.b1 = c->net.be1;
    a.W2T = head ? c->net.WfeT : c->net.We2T; a.b2 = head ? c->net.bfe : c->net.be2;
    a.Ea = head ? c->Gfeat : c->Efeat; a.xa = c->xfeat;
    a.wf2 = c->net.wf2; a.bf2 = c->net.bf2;
    a.m_out = c->mfeat; a.carry_m = c->carry_m; a.Fraw = c->Fraw; a.carry_f = c->carry_f;
    (void)layer;
    if (c->net.K == 32 && c->net.H == 64) return launch_pair_t<32, 64>(c, a, head);
    if (c->net.K == 64 && c->net.H == 128) return launch_pair_t<64, 128>(c, a, head);
    pimd_set_error("unsupported (n_rbf, hidden) = (%d, %d)", c->net.K, c->net.H);
    return PIMD_ERR_ARG;
}

}  // namespace gfn
