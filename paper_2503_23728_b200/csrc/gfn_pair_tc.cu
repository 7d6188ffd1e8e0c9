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
//   -> the second product is formed TRANSPOSED (M = channels, N = pairs), so that in the tcgen05.ld
//      epilogue a thread owns one channel and walks pairs in CSR order: gathers of x_j, E_j are coalesced
//      over channels and the segmented sum of e_ij = e0_ij + E_i + E_j (S:G5) is a private running sum
//      flushed at row boundaries (same carry slots as the fp32 kernel; no floating-point atomics).
// SiLU(x) = h tanh(h) + h with h = x/2: the factor 1/2 is folded (exactly) into the bf16 weight images.
#include "common.cuh"
#include "tc_ptx.cuh"

namespace gfn_tc {

constexpr int TP = 128;      // pairs per tile
constexpr int H = 128;       // channels
constexpr int K = 64;        // radial basis functions
constexpr int GT = 256;      // threads per group
constexpr int NG = 2;        // groups per CTA

struct PairArgs {
    int N, periodic;
    double box[3];
    float r_cut, wscale;
    const int *row_ptr, *col, *pair_row;
    int64_t rows;
    const double *q;
    const uint16_t *W1img, *W2img;        // bf16 UMMA images: 0.5 W_e1 [128][64]; W_e2 (message) or 0.5 W_f1 W_e2 (head), 2 x [128][64]
    const float *b1, *b2;
    const uint32_t *XE;                   // message: packed bf16 (x | E << 16) per (row, channel)
    const float *Gf;                      // head: fp32 G = W_f1 E
    const float *wf2; float bf2;
    float *m_out, *carry_m, *Fraw, *carry_f;
};

struct GroupSmem {
    __align__(1024) unsigned char ops[49152];   // A1 (RBF tile, 16 KB) + A2 (h1, 2 x 16 KB): bf16 UMMA operand tiles
    double d[TP];
    __align__(16) float w[TP];
    __align__(16) int joff[TP];                 // jrow * H
    float u[TP][3], s4[4][TP];
    int row[TP], rs[TP], re[TP];
    unsigned fmask[8];                          // per 16-pair chunk: bit e set = pair starts a new CSR row segment
    __align__(8) uint64_t mbar;
};

struct Smem {
    __align__(1024) unsigned char W1[TP * K * 2];          // 16384
    __align__(1024) unsigned char W2[2 * TP * 64 * 2];     // 32768
    GroupSmem g[NG];
    float b1[H], b2[H], wf2[H];
    uint32_t tmem_base;
};

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// message-pass flush of one finished row segment (granule [g0, g1), global granule index gidx)
__device__ __forceinline__ void flush_m(const PairArgs &a, const GroupSmem &G, int cur, int pfirst, int64_t g0, int64_t g1,
                                        int64_t gidx, int c, float sum)
{
    if (cur < 0) return;
    const int rs = G.rs[pfirst], re = G.re[pfirst];
    if (rs >= g0 && re <= g1) a.m_out[(size_t)cur * H + c] = sum;
    else if (rs < g0) a.carry_m[(size_t)(gidx * 2 + 0) * H + c] = sum;
    else a.carry_m[(size_t)(gidx * 2 + 1) * H + c] = sum;
}

// D2 is TRANSPOSED: TMEM lane = channel c, column = pair.  Thread (c, half) walks the 64 pairs of its granule in
// CSR order, 16 at a time (one tcgen05.ld).  Chunks without a row boundary (fmask == 0) take a branch-free path.
template <bool HEAD>
__device__ __forceinline__ void epilogue(const PairArgs &a, Smem &S, GroupSmem &G, const uint32_t *__restrict__ XE,
                                         const float *__restrict__ Gf, uint32_t tmem_lane, int c, int half, int lane,
                                         int gtid, int64_t tile0, int bar_id)
{
    constexpr int GP = 64;
    const float b2c = S.b2[c];
    if (!HEAD) {
        const int64_t g0 = tile0 + (int64_t)half * GP, g1 = g0 + GP, gidx = g0 / GP;
        int cur = -1, pfirst = 0;
        float sum = 0.f, be = 0.f;
#pragma unroll 1
        for (int cc = 0; cc < 4; ++cc) {
            const int q0 = half * GP + cc * 16;
            float v[16], w[16];
            uint32_t xe[16];
#pragma unroll
            for (int e4 = 0; e4 < 4; ++e4) {
                const int4 o = *(const int4 *)&G.joff[q0 + e4 * 4];
                xe[e4 * 4 + 0] = __ldg(XE + o.x + c); xe[e4 * 4 + 1] = __ldg(XE + o.y + c);
                xe[e4 * 4 + 2] = __ldg(XE + o.z + c); xe[e4 * 4 + 3] = __ldg(XE + o.w + c);
                *(float4 *)&w[e4 * 4] = *(const float4 *)&G.w[q0 + e4 * 4];
            }
            const unsigned mask = G.fmask[half * 4 + cc];
            tc::tmem_ld16(tmem_lane + q0, v);
            if (mask == 0u) {
#pragma unroll
                for (int e = 0; e < 16; ++e)
                    sum = fmaf((v[e] + be) + tc::bf16hi_to_f32(xe[e]), w[e] * tc::bf16lo_to_f32(xe[e]), sum);
            } else {
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    if ((mask >> e) & 1u) {   // warp-uniform
                        flush_m(a, G, cur, pfirst, g0, g1, gidx, c, sum);
                        cur = G.row[q0 + e]; pfirst = q0 + e; sum = 0.f;
                        be = b2c + ((cur >= 0) ? tc::bf16hi_to_f32(__ldg(XE + (size_t)cur * H + c)) : 0.f);
                    }
                    // w = 0 for pairs past the end of the list
                    sum = fmaf((v[e] + be) + tc::bf16hi_to_f32(xe[e]), w[e] * tc::bf16lo_to_f32(xe[e]), sum);
                }
            }
        }
        flush_m(a, G, cur, pfirst, g0, g1, gidx, c, sum);
        tc::tc_fence_before_sync();
    } else {
        // s_p = sum_c w_f2[c] SiLU(t), t = D2 + b_fe + G_i + G_j; here everything is carried as h = t/2.
        // Per-thread term for channel c, then a fixed-tree transposing reduction over the 32 lanes and the 4 quarters.
        const float wc = S.wf2[c];
        const int quarter = (gtid >> 5) & 3;
        float be = 0.f;
#pragma unroll 1
        for (int cc = 0; cc < 4; ++cc) {
            const int q0 = half * GP + cc * 16;
            float v[16], Gj[16];
#pragma unroll
            for (int e4 = 0; e4 < 4; ++e4) {
                const int4 o = *(const int4 *)&G.joff[q0 + e4 * 4];
                Gj[e4 * 4 + 0] = __ldg(Gf + o.x + c); Gj[e4 * 4 + 1] = __ldg(Gf + o.y + c);
                Gj[e4 * 4 + 2] = __ldg(Gf + o.z + c); Gj[e4 * 4 + 3] = __ldg(Gf + o.w + c);
            }
            const unsigned mask = G.fmask[half * 4 + cc];
            tc::tmem_ld16(tmem_lane + q0, v);
            if (mask == 0u) {
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    const float h = fmaf(0.5f, Gj[e], v[e] + be);
                    v[e] = wc * fmaf(h, tc::tanh_approx(h), h);
                }
            } else {
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    if ((mask >> e) & 1u) {
                        const int r = G.row[q0 + e];
                        be = b2c + ((r >= 0) ? 0.5f * __ldg(Gf + (size_t)r * H + c) : 0.f);
                    }
                    const float h = fmaf(0.5f, Gj[e], v[e] + be);
                    v[e] = wc * fmaf(h, tc::tanh_approx(h), h);
                }
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const float send = (lane & 16) ? v[i] : v[i + 8], keep = (lane & 16) ? v[i + 8] : v[i];
                v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float send = (lane & 8) ? v[i] : v[i + 4], keep = (lane & 8) ? v[i + 4] : v[i];
                v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
            }
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const float send = (lane & 4) ? v[i] : v[i + 2], keep = (lane & 4) ? v[i + 2] : v[i];
                v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
            }
            {
                const float send = (lane & 2) ? v[0] : v[1], keep = (lane & 2) ? v[1] : v[0];
                v[0] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
            }
            v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
            // lane bits (4,3,2,1) select pair e = 8 b4 + 4 b3 + 2 b2 + b1
            if ((lane & 1) == 0)
                G.s4[quarter][q0 + ((lane >> 4) & 1) * 8 + ((lane >> 3) & 1) * 4 + ((lane >> 2) & 1) * 2 + ((lane >> 1) & 1)] = v[0];
        }
        tc::tc_fence_before_sync();
        tc::named_bar_sync(bar_id, GT);
        if (gtid < TP) {
            const int key = G.row[gtid];
            const float f = G.w[gtid] * (((G.s4[0][gtid] + G.s4[1][gtid]) + (G.s4[2][gtid] + G.s4[3][gtid])) + a.bf2);
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
}

template <bool HEAD>
__global__ void __launch_bounds__(GT * NG, 1) pair_tc_kernel(const __grid_constant__ PairArgs a)
{
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    // keep the shared state space visible to the compiler (LDS/STS, not generic LD/ST)
    Smem &S = *reinterpret_cast<Smem *>(smem_raw + ((1024u - (tc::smem_u32(smem_raw) & 1023u)) & 1023u));
    const int tid = threadIdx.x, grp = tid / GT, gtid = tid % GT, warp = tid >> 5, lane = tid & 31;
    const int64_t n_pairs = a.row_ptr[a.rows];
    if ((int64_t)blockIdx.x * (NG * TP) >= n_pairs) return;   // uniform per CTA
    GroupSmem &G = S.g[grp];
    const uint32_t *__restrict__ XE = a.XE;
    const float *__restrict__ Gf = a.Gf;

    // ---- one-time setup: weights (generic proxy) -> smem, mbarriers, TMEM
    {
        const uint4 *s1 = (const uint4 *)a.W1img, *s2 = (const uint4 *)a.W2img;
        uint4 *d1 = (uint4 *)S.W1, *d2 = (uint4 *)S.W2;
        for (int i = tid; i < TP * K * 2 / 16; i += GT * NG) d1[i] = __ldg(s1 + i);
        for (int i = tid; i < 2 * TP * 64 * 2 / 16; i += GT * NG) d2[i] = __ldg(s2 + i);
        for (int i = tid; i < H; i += GT * NG) {
            S.b1[i] = 0.5f * a.b1[i];
            S.b2[i] = HEAD ? 0.5f * a.b2[i] : a.b2[i];
            S.wf2[i] = HEAD ? a.wf2[i] : 0.f;
        }
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
    const int p = gtid & 127, half = gtid >> 7;                // pair (TMEM lane of D1) / channel (lane of D2^T); column half
    const uint32_t lane_field = (uint32_t)(p & ~31) << 16;      // TMEM lane base of this warp: 32 * (warp % 4)
    const double inv_delta = (double)(K - 1) / (double)a.r_cut;
    const int bar_id = 1 + grp;
    uint32_t parity = 0;
    constexpr float RBF_C = 0.84932180028801904f;               // sqrt(0.5 log2 e): exp(-t^2/2) = 2^-(C t)^2

    for (int64_t tile0 = ((int64_t)blockIdx.x * NG + grp) * TP; tile0 < n_pairs; tile0 += (int64_t)gridDim.x * NG * TP) {
        // ---- per-pair geometry (S:G1), fp64 minimum image; row-segment flags
        if (gtid < TP) {
            const int64_t pg = tile0 + gtid;
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
            int prev = __shfl_up_sync(0xffffffffu, row, 1);
            if (lane == 0) prev = ((gtid & 63) == 0) ? -2 : ((pg - 1 < n_pairs) ? a.pair_row[pg - 1] : -1);
            const unsigned fm = __ballot_sync(0xffffffffu, row != prev);
            if (lane == 0) { G.fmask[2 * (gtid >> 5)] = fm & 0xFFFFu; G.fmask[2 * (gtid >> 5) + 1] = fm >> 16; }
            G.row[gtid] = row; G.joff[gtid] = jrow * H; G.rs[gtid] = rs; G.re[gtid] = re;
            G.d[gtid] = dist; G.w[gtid] = w; G.u[gtid][0] = ux; G.u[gtid][1] = uy; G.u[gtid][2] = uz;
        }
        tc::named_bar_sync(bar_id, GT);
        // ---- RBF tile -> A1 (bf16, K-major rows of 128 B, 16-byte chunks XOR-swizzled by row & 7)
        {
            const float uc = (float)(G.d[p] * inv_delta) * RBF_C;   // C d / delta
#pragma unroll
            for (int ci = 0; ci < 4; ++ci) {
                const int ch = half * 4 + ci;
                float g[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const float t = uc - RBF_C * (float)(ch * 8 + e);
                    g[e] = ex2_approx(-t * t);
                }
                uint4 v = make_uint4(tc::pack_bf16(g[0], g[1]), tc::pack_bf16(g[2], g[3]), tc::pack_bf16(g[4], g[5]),
                                     tc::pack_bf16(g[6], g[7]));
                *(uint4 *)(A1 + p * 128 + ((ch ^ (p & 7)) << 4)) = v;
            }
        }
        tc::fence_proxy_async_smem();
        tc::named_bar_sync(bar_id, GT);
        // ---- D1 = G . (W_e1/2)^T   (4 x UMMA 128x128x16)
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
        // ---- h1 = SiLU(2 (D1 + b_e1/2)) -> A2 (this thread: its pair's 64 columns of K-block `half`)
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
            float v[16];
            tc::tmem_ld16(tmem_d1 + lane_field + half * 64 + cc * 16, v);
            uint32_t pk[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const int col = half * 64 + cc * 16 + 2 * e;
                const float h0 = v[2 * e] + S.b1[col], h1 = v[2 * e + 1] + S.b1[col + 1];
                pk[e] = tc::pack_bf16(fmaf(h0, tc::tanh_approx(h0), h0), fmaf(h1, tc::tanh_approx(h1), h1));
            }
            unsigned char *rowp = A2 + half * 16384 + p * 128;
            *(uint4 *)(rowp + (((cc * 2) ^ (p & 7)) << 4)) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
            *(uint4 *)(rowp + (((cc * 2 + 1) ^ (p & 7)) << 4)) = make_uint4(pk[4], pk[5], pk[6], pk[7]);
        }
        tc::tc_fence_before_sync();
        tc::fence_proxy_async_smem();
        tc::named_bar_sync(bar_id, GT);
        // ---- D2^T = W2 . h1^T   (8 x UMMA 128x128x16; M = channels, N = pairs)
        if (gtid == 0) {
            tc::tc_fence_after_sync();
#pragma unroll
            for (int kk = 0; kk < H / 16; ++kk) {
                const uint32_t off = (kk >> 2) * 16384 + (kk & 3) * 32;
                tc::mma_bf16_ss(tmem_d2, tc::make_desc_sw128(sW2 + off), tc::make_desc_sw128(sA2 + off), idesc, kk > 0);
            }
            tc::mma_commit(&G.mbar);
        }
        tc::mbar_wait(&G.mbar, parity);
        parity ^= 1;
        tc::tc_fence_after_sync();
        // EPILOGUE (see part 2)
        epilogue<HEAD>(a, S, G, XE, Gf, tmem_d2 + lane_field, p, half, lane, gtid, tile0, bar_id);
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
    a.XE = c->XE; a.Gf = c->Gfeat;
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
