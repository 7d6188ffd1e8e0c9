// gfn_pair_tc.cu -- fused per-pair kernels of the GFN force net on the 5th-gen tensor cores
// (rows a5, a7 of SURVEY 8(a)), bf16 operands + fp32 accumulation in TMEM.
// Used when gemm_dtype == 1 and (K, H) == (64, 128)  (BASELINE configs[3..4]; tolerance 2e-2).
//
// One persistent CTA per SM holds the bf16 filter weights (W_e1, and W_e2 or W_f1 W_e2) in shared
// memory once, pre-swizzled for UMMA (K-major, 128-byte swizzle).  Two independent 256-thread groups
// share them and ping-pong over 128-pair tiles of the flat CSR pair list, each with its own operand
// buffers, mbarrier and 256 TMEM columns, synchronising with named barriers only, so one group's
// MUFU/epilogue work overlaps the other group's MMAs.  Per tile:
//   fp64 geometry -> Gaussian RBF tile (bf16, swizzled smem) -> tcgen05.mma 128x128x64 -> TMEM
//   -> tcgen05.ld, +bias, SiLU, bf16 -> swizzled smem -> tcgen05.mma 128x128x128 -> TMEM
//   -> tcgen05.ld epilogue with e_ij = e0_ij + E_i + E_j (S:G5) and the same deterministic
//      segmented reductions / carry slots as the fp32 kernel (no floating-point atomics).
#include "common.cuh"
#include "tc_ptx.cuh"

namespace gfn_tc {

constexpr int TP = 128;      // pairs per tile (UMMA M)
constexpr int H = 128;       // channels (UMMA N)
constexpr int K = 64;        // radial basis functions
constexpr int GT = 256;      // threads per group
constexpr int NG = 2;        // groups per CTA
constexpr int VSTRIDE = 132; // fp32 row stride of the message tile (conflict-free float4 stores)

struct PairArgs {
    int N, periodic;
    double box[3];
    float r_cut, wscale;
    const int *row_ptr, *col, *pair_row;
    int64_t rows;
    const double *q;
    const uint16_t *W1img, *W2img;        // bf16, pre-swizzled UMMA images: [128][64] and 2 x [128][64]
    const float *b1, *b2;
    const float *Ea, *xa;                 // message: E, x ; head: G, unused
    const float *wf2; float bf2;
    float *m_out, *carry_m, *Fraw, *carry_f;
};

struct GroupSmem {
    // A1 (RBF tile, 16 KB) and A2 (2 x 16 KB) are dead once the second MMA has completed; the fp32
    // message tile [TP][VSTRIDE] is laid over them and the tail.
    __align__(1024) unsigned char ops[TP * VSTRIDE * 4];   // 67584 B >= 49152
    double d[TP];
    float w[TP], u[TP][3], s2[2][TP];
    int row[TP], jrow[TP], rs[TP], re[TP];
    __align__(8) uint64_t mbar;
};

struct Smem {
    __align__(1024) unsigned char W1[TP * K * 2];          // 16384
    __align__(1024) unsigned char W2[2 * TP * 64 * 2];     // 32768
    GroupSmem g[NG];
    float b1[H], b2[H], wf2[H];
    uint32_t tmem_base;
};

template <bool HEAD>
__global__ void __launch_bounds__(GT * NG, 1) pair_tc_kernel(PairArgs a)
{
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    Smem &S = *reinterpret_cast<Smem *>((((uintptr_t)smem_raw) + 1023) & ~(uintptr_t)1023);
    const int tid = threadIdx.x, grp = tid / GT, gtid = tid % GT, warp = tid >> 5;
    const int64_t n_pairs = a.row_ptr[a.rows];
    if ((int64_t)blockIdx.x * (NG * TP) >= n_pairs) return;   // uniform per CTA
    GroupSmem &G = S.g[grp];

    // ---- one-time setup: weights (generic proxy) -> smem, mbarriers, TMEM
    {
        const uint4 *s1 = (const uint4 *)a.W1img, *s2 = (const uint4 *)a.W2img;
        uint4 *d1 = (uint4 *)S.W1, *d2 = (uint4 *)S.W2;
        for (int i = tid; i < TP * K * 2 / 16; i += GT * NG) d1[i] = __ldg(s1 + i);
        for (int i = tid; i < 2 * TP * 64 * 2 / 16; i += GT * NG) d2[i] = __ldg(s2 + i);
        for (int i = tid; i < H; i += GT * NG) { S.b1[i] = a.b1[i]; S.b2[i] = a.b2[i]; S.wf2[i] = HEAD ? a.wf2[i] : 0.f; }
        if (gtid == 0) tc::mbar_init(&G.mbar, 1);
        if (warp == 0) tc::tmem_alloc(&S.tmem_base, 512);
        tc::fence_mbar_init();
        tc::fence_proxy_async_smem();
        tc::tc_fence_before_sync();
        __syncthreads();
        tc::tc_fence_after_sync();
    }
    const uint32_t tmem_d1 = S.tmem_base + grp * 256, tmem_d2 = tmem_d1 + 128;
    const uint32_t idesc = tc::make_idesc_bf16(TP, H);
    const uint32_t sW1 = tc::smem_u32(S.W1), sW2 = tc::smem_u32(S.W2);
    unsigned char *A1 = G.ops, *A2 = G.ops + 16384;
    const uint32_t sA1 = tc::smem_u32(A1), sA2 = tc::smem_u32(A2);
    float *vt = reinterpret_cast<float *>(G.ops);
    const int p = gtid & 127, half = gtid >> 7;                // this thread's pair (TMEM lane) and column half
    const uint32_t lane_field = (uint32_t)(p & ~31) << 16;      // TMEM lane base of this warp: 32 * (warp % 4)
    const double inv_delta = (double)(K - 1) / (double)a.r_cut;
    const int bar_id = 1 + grp;
    uint32_t parity = 0;

    for (int64_t tile0 = ((int64_t)blockIdx.x * NG + grp) * TP; tile0 < n_pairs; tile0 += (int64_t)gridDim.x * NG * TP) {
        // ---- per-pair geometry (S:G1), fp64 minimum image
        if (gtid < TP) {
            int64_t pg = tile0 + gtid;
            int row = -1, jrow = 0, rs = 0, re = 0;
            double dist = 0.0;
            float w = 0.f, ux = 0.f, uy = 0.f, uz = 0.f;
            if (pg < n_pairs) {
                row = a.pair_row[pg];
                int sys = row / a.N;
                jrow = sys * a.N + a.col[pg];
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
            G.row[gtid] = row; G.jrow[gtid] = jrow; G.rs[gtid] = rs; G.re[gtid] = re;
            G.d[gtid] = dist; G.w[gtid] = w; G.u[gtid][0] = ux; G.u[gtid][1] = uy; G.u[gtid][2] = uz;
        }
        tc::named_bar_sync(bar_id, GT);
        // ---- RBF tile -> A1 (bf16, K-major rows of 128 B, 16-byte chunks XOR-swizzled by row & 7)
        {
            const float uu = (float)(G.d[p] * inv_delta);   // d / delta in fp64, then fp32
#pragma unroll
            for (int ci = 0; ci < 4; ++ci) {
                const int c = half * 4 + ci;
                float g[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    float t = uu - (float)(c * 8 + e);
                    g[e] = __expf(-0.5f * t * t);
                }
                uint4 v = make_uint4(tc::pack_bf16(g[0], g[1]), tc::pack_bf16(g[2], g[3]), tc::pack_bf16(g[4], g[5]),
                                     tc::pack_bf16(g[6], g[7]));
                *(uint4 *)(A1 + p * 128 + ((c ^ (p & 7)) << 4)) = v;
            }
        }
        tc::fence_proxy_async_smem();
        tc::named_bar_sync(bar_id, GT);
        // ---- D1 = G . W_e1^T   (4 x UMMA 128x128x16)
        if (gtid == 0) {
            tc::tc_fence_after_sync();
#pragma unroll
            for (int kk = 0; kk < K / 16; ++kk)
                tc::mma_bf16_ss(tmem_d1, tc::make_desc_sw128(sA1 + kk * 32), tc::make_desc_sw128(sW1 + kk * 32), idesc, kk > 0);
            tc::mma_commit(&G.mbar);
        }
        tc::mbar_wait(&G.mbar, parity);
        parity ^= 1;
        tc::tc_fence_after_sync();
        // ---- h1 = SiLU(D1 + b_e1) -> A2 (this thread: its pair's 64 columns of K-block `half`)
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
            float v[16];
            tc::tmem_ld16(tmem_d1 + lane_field + half * 64 + cc * 16, v);
            uint32_t pk[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const int col = half * 64 + cc * 16 + 2 * e;
                pk[e] = tc::pack_bf16(tc::silu_tanh(v[2 * e] + S.b1[col]), tc::silu_tanh(v[2 * e + 1] + S.b1[col + 1]));
            }
            unsigned char *rowp = A2 + half * 16384 + p * 128;
            *(uint4 *)(rowp + (((cc * 2) ^ (p & 7)) << 4)) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
            *(uint4 *)(rowp + (((cc * 2 + 1) ^ (p & 7)) << 4)) = make_uint4(pk[4], pk[5], pk[6], pk[7]);
        }
        tc::tc_fence_before_sync();
        tc::fence_proxy_async_smem();
        tc::named_bar_sync(bar_id, GT);
        // ---- D2 = h1 . W2^T   (8 x UMMA 128x128x16)
        if (gtid == 0) {
            tc::tc_fence_after_sync();
#pragma unroll
            for (int kk = 0; kk < H / 16; ++kk) {
                const uint32_t off = (kk >> 2) * 16384 + (kk & 3) * 32;
                tc::mma_bf16_ss(tmem_d2, tc::make_desc_sw128(sA2 + off), tc::make_desc_sw128(sW2 + off), idesc, kk > 0);
            }
            tc::mma_commit(&G.mbar);
        }
        tc::mbar_wait(&G.mbar, parity);
        parity ^= 1;
        tc::tc_fence_after_sync();

        const int row = G.row[p], jrow = G.jrow[p];
        if (!HEAD) {
            // val[p][c] = w_p (e0 + E_i + E_j)[c] x_j[c]  -> message tile (fp32, row stride VSTRIDE)
            const float w = G.w[p];
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) {
                const int c0 = half * 64 + cc * 16;
                float v[16];
                tc::tmem_ld16(tmem_d2 + lane_field + c0, v);
                if (row >= 0) {
#pragma unroll
                    for (int q4 = 0; q4 < 4; ++q4) {
                        const int c = c0 + q4 * 4;
                        float4 Ei = __ldg((const float4 *)(a.Ea + (size_t)row * H + c));
                        float4 Ej = __ldg((const float4 *)(a.Ea + (size_t)jrow * H + c));
                        float4 xj = __ldg((const float4 *)(a.xa + (size_t)jrow * H + c));
                        v[q4 * 4 + 0] = w * (v[q4 * 4 + 0] + S.b2[c + 0] + Ei.x + Ej.x) * xj.x;
                        v[q4 * 4 + 1] = w * (v[q4 * 4 + 1] + S.b2[c + 1] + Ei.y + Ej.y) * xj.y;
                        v[q4 * 4 + 2] = w * (v[q4 * 4 + 2] + S.b2[c + 2] + Ei.z + Ej.z) * xj.z;
                        v[q4 * 4 + 3] = w * (v[q4 * 4 + 3] + S.b2[c + 3] + Ei.w + Ej.w) * xj.w;
                    }
                }
                // all MMAs that read A1/A2 have completed (commit observed): the tile may overwrite them
#pragma unroll
                for (int q4 = 0; q4 < 4; ++q4)
                    *(float4 *)&vt[p * VSTRIDE + c0 + q4 * 4] = make_float4(v[q4 * 4], v[q4 * 4 + 1], v[q4 * 4 + 2], v[q4 * 4 + 3]);
            }
            tc::tc_fence_before_sync();
            tc::named_bar_sync(bar_id, GT);
            // deterministic segmented sum: thread (part, ch) walks its 64-pair granule in CSR order
            {
                constexpr int GP = 64;
                const int ch = gtid & 127, part = gtid >> 7;
                const int64_t g0 = tile0 + (int64_t)part * GP, g1 = g0 + GP, gidx = g0 / GP;
                int cur = -1, pfirst = 0;
                float sum = 0.f;
                for (int pp = 0; pp <= GP; ++pp) {
                    const int q = part * GP + pp;
                    const int r = (pp < GP) ? G.row[q] : -2;
                    if (r != cur) {
                        if (cur >= 0) {
                            const int rs = G.rs[pfirst], re = G.re[pfirst];
                            if (rs >= g0 && re <= g1) a.m_out[(size_t)cur * H + ch] = sum;
                            else if (rs < g0) a.carry_m[(size_t)(gidx * 2 + 0) * H + ch] = sum;
                            else a.carry_m[(size_t)(gidx * 2 + 1) * H + ch] = sum;
                        }
                        cur = r; pfirst = q; sum = 0.f;
                    }
                    if (r >= 0) sum += vt[q * VSTRIDE + ch];
                }
            }
        } else {
            // s_p = w_f2 . SiLU(D2 + b_fe + G_i + G_j) + b_f2 ; this thread sums its 64 columns
            float s = 0.f;
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) {
                const int c0 = half * 64 + cc * 16;
                float v[16];
                tc::tmem_ld16(tmem_d2 + lane_field + c0, v);
                if (row >= 0) {
#pragma unroll
                    for (int q4 = 0; q4 < 4; ++q4) {
                        const int c = c0 + q4 * 4;
                        float4 Gi = __ldg((const float4 *)(a.Ea + (size_t)row * H + c));
                        float4 Gj = __ldg((const float4 *)(a.Ea + (size_t)jrow * H + c));
                        s += S.wf2[c + 0] * tc::silu_tanh(v[q4 * 4 + 0] + S.b2[c + 0] + Gi.x + Gj.x);
                        s += S.wf2[c + 1] * tc::silu_tanh(v[q4 * 4 + 1] + S.b2[c + 1] + Gi.y + Gj.y);
                        s += S.wf2[c + 2] * tc::silu_tanh(v[q4 * 4 + 2] + S.b2[c + 2] + Gi.z + Gj.z);
                        s += S.wf2[c + 3] * tc::silu_tanh(v[q4 * 4 + 3] + S.b2[c + 3] + Gi.w + Gj.w);
                    }
                }
            }
            G.s2[half][p] = s;
            tc::tc_fence_before_sync();
            tc::named_bar_sync(bar_id, GT);
            if (gtid < TP) {
                const int lane = gtid & 31;
                const int key = G.row[gtid];
                const float f = G.w[gtid] * (G.s2[0][gtid] + G.s2[1][gtid] + a.bf2);
                float v[3] = {f * G.u[gtid][0], f * G.u[gtid][1], f * G.u[gtid][2]};
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
                    const int64_t g0 = tile0 + (gtid & ~31), g1 = g0 + 32, gidx = g0 >> 5;
                    const int rs = G.rs[gtid], re = G.re[gtid];
                    float *dst;
                    if (rs >= g0 && re <= g1) dst = a.Fraw + (size_t)key * 4;
                    else if (rs < g0) dst = a.carry_f + (size_t)(gidx * 2 + 0) * 4;
                    else dst = a.carry_f + (size_t)(gidx * 2 + 1) * 4;
                    dst[0] = v[0]; dst[1] = v[1]; dst[2] = v[2];
                }
            }
        }
        tc::named_bar_sync(bar_id, GT);   // tile buffers free for the next iteration
    }
    // ---- teardown
    tc::tc_fence_before_sync();
    __syncthreads();
    if (warp == 0) tc::tmem_dealloc(S.tmem_base, 512);
}

int launch_pair_tc(pimd_ctx *c, bool head)
{
    PairArgs a;
    a.N = c->N; a.periodic = c->periodic;
    for (int k = 0; k < 3; ++k) a.box[k] = c->box[k];
    a.r_cut = c->net.r_cut; a.wscale = head ? 1.0f : c->net.agg_norm;
    a.row_ptr = c->nl.row_ptr; a.col = c->nl.col; a.pair_row = c->nl.pair_row; a.rows = c->rows; a.q = c->q;
    a.W1img = c->wimg_e1; a.W2img = head ? c->wimg_fe : c->wimg_e2;
    a.b1 = c->net.be1; a.b2 = head ? c->net.bfe : c->net.be2;
    a.Ea = head ? c->Gfeat : c->Efeat; a.xa = c->xfeat;
    a.wf2 = c->net.wf2; a.bf2 = c->net.bf2;
    a.m_out = c->mfeat; a.carry_m = c->carry_m; a.Fraw = c->Fraw; a.carry_f = c->carry_f;
    const size_t smem = sizeof(Smem) + 1024;
    static bool attr = false;
    if (!attr) {
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(pair_tc_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(pair_tc_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr = true;
    }
    if (head) pair_tc_kernel<true><<<c->num_sms, GT * NG, smem, c->stream>>>(a);
    else pair_tc_kernel<false><<<c->num_sms, GT * NG, smem, c->stream>>>(a);
    c->launches++;
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}

}  // namespace gfn_tc
