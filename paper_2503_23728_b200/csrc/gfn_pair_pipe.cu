// gfn_pair_pipe.cu -- fused per-pair kernels of the GFN force net on the 5th-gen tensor cores, as a
// warp-specialised pipeline (rows a5, a7 of SURVEY 8(a)).  bf16 operands, fp32 accumulation
// in TMEM.  Used when gemm_dtype == 1 and (K, H) == (64, 128)  (BASELINE configs[3..4]; tolerance 2e-2).
//
// One persistent CTA per SM walks 128-pair tiles of the flat CSR pair list.  The roles below run concurrently on
// different tiles and hand buffers to each other through mbarriers and named barriers only (no CTA-wide barrier in the loop).
// First pair pass of a force evaluation (MODE 0):
//   P   4 warps, thread = pair : row, column, displacement r_j - r_i and segment kind streamed from the neighbour list (the fill
//                                kernel forms the fp64 minimum-image difference) -> distance, cutoff weight, row-segment flags (meta ring);
//                                Gaussian RBF tile -> A1 (bf16, K-major, 128-byte swizzle)
//   MMA 1 thread               : D1 = A1 (W_e1/2)^T  (4 x UMMA 128x128x16);  D2^T = W2 A2^T  (8 x UMMA), W2 = W_e2 or W_f1 W_e2/2
//   H   4 warps, thread = pair : D1 (TMEM) + b -> SiLU -> A2 (bf16 operand of the second product)
//   S   1 warp                 : TMA bulk stores of the tile's A2 image (32 KB) and meta record to HBM
//   G   4 warps                : TMA tile::gather4 copies of the gathered rows (x_j, y_j = E_j x_j in one word, or G_j fp32; 4 x 512 B per copy)
//                                into an 8-slot shared-memory ring, 16 pairs per slot
//   E   16 warps, thread = (channel, quarter tile): D2^T (TMEM lane = channel) -> e_ij = e0_ij + E_i + E_j (S:G5) ->
//                                private running sums over CSR row segments, cut at row boundaries.
// The filter's first layer does not depend on the interaction layer, so the later passes (MODE 1: remaining message
// passes and the force head) replace P, H and the first product by
//   L   1 warp                 : two TMA bulk copies per tile bring the A2 image and the meta record back
// and the head runs its channel reduction on the tensor core:
//   E   (head)                 : act = SiLU(W_fe h1 + b_fe + G_i + G_j) written as a bf16 MN-major operand A3 (pairs contiguous)
//   MMA                        : D3[p][.] = act[p][:] . w_f2   (8 x UMMA 128x16x16)
//   F   4 warps, thread = pair : s_p from D3 -> c_ij s_ij u_ij, segmented warp scan over 32-pair granules -> forces.
// (When L = 0 the head is the first pass; it then reduces over channels with a fixed shuffle tree.)
// Waiting: mbarrier try_wait does not suspend on this part (it polls, and every poll takes an issue slot from the warps
// that have work).  So per role ONE warp polls the mbarriers that tensor-core commits and TMA transactions complete
// on, and releases its role's other warps through a named barrier (bar.sync blocks in hardware); the pollers sit on
// different SM sub-partitions.  Hand-offs between threads only (ring slot consumed: E -> G) are named barriers.
// Row segments that straddle a reduction granule go through carry slots that the consumer adds in a fixed
// order: no floating-point atomics, bitwise reproducible.
// SiLU(x) = h tanh(h) + h with h = x/2: the factor 1/2 is folded (exactly) into the bf16 weight images.
#include "common.cuh"
#include "tc_ptx.cuh"
#ifdef GFN_PIPE_STATS
#include <stdio.h>
#endif

namespace gfn_pipe {

// -DGFN_PIPE_STATS: every role counts the cycles it spends waiting; block 0 prints them (diagnostic builds only)
#ifdef GFN_PIPE_STATS
#define WAITED(stmt)                       \
    do {                                   \
        const long long t0_ = clock64();   \
        stmt;                              \
        g_wait_ += clock64() - t0_;        \
    } while (0)
#define STATS_BEGIN long long g_wait_ = 0; long long g_wk_[4] = {0, 0, 0, 0}; const long long g_start_ = clock64();
#define WAITEDK(k, stmt)                   \
    do {                                   \
        const long long t0_ = clock64();   \
        stmt;                              \
        g_wk_[k] += clock64() - t0_;       \
        g_wait_ += clock64() - t0_;        \
    } while (0)
#define STATS_END(name)                                                                                              \
    if (blockIdx.x == 0 && (threadIdx.x & 31) == 0)                                                                  \
        printf("%s warp %2d: total %lld cycles, waiting %lld (%.0f%%) [%lld %lld %lld %lld]\n", name, (int)(threadIdx.x >> 5), clock64() - g_start_, \
               g_wait_, 100.0 * g_wait_ / (double)(clock64() - g_start_), g_wk_[0], g_wk_[1], g_wk_[2], g_wk_[3]);
#else
#define WAITED(stmt) stmt
#define WAITEDK(k, stmt) stmt
#define STATS_BEGIN
#define STATS_END(name)
#endif

// wait of a role that is idle most of the time (the MMA thread, the store warp S): polls at the pace of an L2 round trip (tc_ptx.cuh).
// The polled word is any readable one, a different 32-byte sector per CTA; the scratch word is never read.
#define LAZY_WAIT(barp, par) tc::mbar_wait_lazy(barp, par, a.h1_img + (size_t)blockIdx.x * 32, S + OFF_TMEM + 8)

constexpr int TP = 128;      // pairs per tile
constexpr int H = 128;       // channels
constexpr int K = 64;        // radial basis functions
constexpr int NM = 4;        // meta ring depth (tiles)
constexpr int NSLOT = 4;     // quarter tiles; the gather ring has two 16-pair slots per quarter
// Warp layout per kernel variant (fewer warps in the later passes -> more registers per thread for role E):
//   MODE 0           : P 0-3, H 4-7, E 8-23, MMA 24, G 25-28, S 29, idle 30-31 (32 warps, 64 registers at launch; setmaxnreg
//                      moves registers from the P, H, MMA/G/S warpgroups (56, 56, 40) to the four E warpgroups (80))
//   MODE 1, message  : E 0-15, G 16-19, MMA 20, L 21                          (22 warps, 80 registers used)
//   MODE 1, head     : E 0-15, F 16-19, G 20-23, MMA 24, L 25, idle 26-27     (28 warps, 72 at launch; setmaxnreg: E 88, F 56, rest 40)
// E and F/H warps start at a multiple of 4: warp % 4 is the TMEM lane quadrant a warp may access.
template <bool HEAD, int MODE>
struct Warps {
    static constexpr int E0 = (MODE == 0) ? 8 : 0;
    static constexpr int F0 = (MODE == 0) ? 4 : 16;                      // H (MODE 0) or F (MODE 1 head)
    static constexpr int G0 = (MODE == 0) ? 25 : (HEAD ? 20 : 16);
    static constexpr int MMA = (MODE == 0) ? 24 : (HEAD ? 24 : 20);
    static constexpr int SL = (MODE == 0) ? 29 : MMA + 1;                // S (MODE 0) or L (MODE 1)
    static constexpr int N = (MODE == 0) ? 32 : (HEAD ? 28 : SL + 1);    // whole warpgroups where setmaxnreg is used; the last warps are idle
    static constexpr int THREADS = N * 32;
};

struct PairArgs {
    alignas(64) CUtensorMap gmap;         // the gathered table (XE or G) as a 2-D tensor [rows][128 x 32 bit] for TMA tile::gather4
    int N;
    float r_cut, wscale;
    const int *row_ptr, *col, *pair_row;
    const float4 *dvec;                   // per pair: r_j - r_i (fp32 of the fp64 minimum-image difference) | segment kind (nlist_kernels.cu)
    int64_t rows;
    const uint16_t *Wf2img;               // head: bf16 UMMA image of w_f2 replicated on 16 rows ([16][128], 4 KB)
    const uint16_t *W1img, *W2img;        // bf16 UMMA images: 0.5 W_e1 [128][64]; W_e2 (message) or 0.5 W_f1 W_e2 (head), 2 x [128][64]
    float b1h[H];                         // b_e1 / 2 (kernel-parameter constant bank: immediate operands in role H)
    const float *b2;
    const void *gsrc;                     // message: XE [rows][128] u32, x bf16 in the low half, the word as fp32 = y = E x (tc::pack_x_y); head: G fp32 [rows][128]
    const float *Emaster;                 // message: fp32 master of E, tile-blocked (gfn_node_tc.cu), for E_i
    const float *wf2; float bf2;
    float *m_out, *carry_m, *Fraw, *carry_f;
    unsigned char *h1_img, *meta_img;     // per tile: A2 operand image (32 KB) and Meta, written by the first pass of a force
                                          // evaluation and re-read by the later ones (same pairs, same h1)
};

struct Meta {
    float w[TP];                 // cutoff weight c_ij (0 for pairs past the end of the list)
    int jrow[TP];                // global row of atom j
    int rowk[TP];                // global row of atom i | kind << 29;  -1 past the end of the list
    float u[3][TP];              // unit vector (r_i - r_j)/d  (head)
    unsigned fmask[8];           // per 16-pair chunk: bit e set = pair starts a new row segment
};

static_assert(sizeof(Meta) == 3104 && sizeof(Meta) % 16 == 0, "Meta is copied by TMA bulk copies; pimd_api.cu sizes meta_img with 3104");

// shared-memory carve (offsets from a 1024-aligned base)
constexpr int OFF_W1 = 0;                          // 16 KB
constexpr int OFF_W2 = OFF_W1 + 16384;             // 32 KB
constexpr int OFF_A1 = OFF_W2 + 32768;             // 2 x 16 KB
constexpr int OFF_A2 = OFF_A1 + 2 * 16384;         // 2 x 32 KB
constexpr int OFF_RING = OFF_A2 + 2 * 32768;       // 4 x 16 KB
constexpr int OFF_META = OFF_RING + NSLOT * 16384; // NM x sizeof(Meta)
constexpr int OFF_BIAS = OFF_META + NM * (int)sizeof(Meta);   // b1, b2, wf2
constexpr int OFF_S4 = OFF_BIAS + 3 * H * 4;       // head: s4[4][TP]
constexpr int OFF_BAR = OFF_S4 + 4 * TP * 4;
constexpr int N_BAR = 76;
constexpr int OFF_TMEM = OFF_BAR + N_BAR * 8;
constexpr int SMEM_BYTES = OFF_TMEM + 16;

// named barriers (0 is __syncthreads)
enum { NB_P = 1, NB_H = 2, NB_E = 3 /* +quarter */, NB_S4 = 7, NB_SLOT = 8 /* +slot: ring slot consumed, E (128) -> G (32) */ };

// mbarrier indices
enum { A1_FULL = 0, A1_EMPTY = 2, D1_FULL = 4, D1_EMPTY = 6, A2_FULL = 8, A2_EMPTY = 10, D2_FULL = 12, D2_EMPTY = 14,
       XE_FULL = 16, META_FULL = 24, META_EMPTY = 28, W_FULL = 32, A3_FULL = 33, A3_EMPTY = 35, D3_FULL = 37, D3_EMPTY = 39 };

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ int n_my_tiles(int64_t n_pairs)
{
    const int64_t n_tiles = (n_pairs + TP - 1) / TP;
    if ((int64_t)blockIdx.x >= n_tiles) return 0;
    return (int)((n_tiles - 1 - blockIdx.x) / gridDim.x) + 1;
}

// kind of the segment of row [rs, re) inside the granule [g0, g0 + GP): 0 whole row here (direct store),
// 1 row began in an earlier granule (carry slot 0), 2 row continues into a later granule (carry slot 1)
__device__ __forceinline__ int seg_kind(int rs, int re, int64_t g0, int GP)
{
    if (rs >= g0 && re <= g0 + GP) return 0;
    return (rs < g0) ? 1 : 2;
}

__device__ __forceinline__ Meta &meta_of(unsigned char *S, int it) { return *(Meta *)(S + OFF_META + (it & (NM - 1)) * (int)sizeof(Meta)); }

constexpr float RBF_C = 0.84932180028801904f;   // sqrt(0.5 log2 e): exp(-t^2/2) = 2^-(C t)^2
constexpr unsigned FULL = 0xffffffffu;

// ---- role P: per-pair geometry (S:G1) + Gaussian RBF tile.  Thread p owns pair p of every tile of this CTA.
template <bool HEAD>
__device__ __forceinline__ void role_P(const PairArgs &a, unsigned char *S, uint64_t *bar, int n_my, int64_t n_pairs, int p,
                                       int lane)
{
    STATS_BEGIN
    constexpr int GP = 32;                        // pairs per reduction granule of the consumer (a quarter tile)
    const float inv_rc = 1.0f / a.r_cut;
    const float uc_scale = (float)(K - 1) / a.r_cut * RBF_C;
    const int64_t stride = (int64_t)gridDim.x * TP;
    int64_t pg = (int64_t)blockIdx.x * TP + p;
    // everything role P needs of a pair is streamed, coalesced, one tile ahead: row, column, and the displacement r_j - r_i with
    // the row's segment kind (written by the neighbour-list fill kernel: no dependent loads behind the indices)
    int row_n = -1, col_n = 0;
    float4 dv_n = make_float4(0.f, 0.f, 0.f, 0.f);
    if (n_my > 0 && pg < n_pairs) { row_n = __ldg(a.pair_row + pg); col_n = __ldg(a.col + pg); dv_n = __ldg(a.dvec + pg); }
    for (int it = 0; it < n_my; ++it, pg += stride) {
        const int row = row_n, cj = col_n;
        const float4 dv = dv_n;
        if (it + 1 < n_my) {                      // the next tile: in flight during this tile's arithmetic
            const int64_t pn = pg + stride;
            row_n = -1; col_n = 0;
            if (pn < n_pairs) { row_n = __ldg(a.pair_row + pn); col_n = __ldg(a.col + pn); dv_n = __ldg(a.dvec + pn); }
        }
        int jrow = 0, kind = 0;
        float w = 0.f, ux = 0.f, uy = 0.f, uz = 0.f, dist = 0.f;
        if (row >= 0) {
            const int sys = row / a.N;
            jrow = sys * a.N + cj;
            const float d2 = fmaf(dv.x, dv.x, fmaf(dv.y, dv.y, dv.z * dv.z));
            const float inv = rsqrtf(fmaxf(d2, 1e-24f));
            dist = d2 * inv;
            ux = -dv.x * inv; uy = -dv.y * inv; uz = -dv.z * inv;
            w = 0.5f * (cospif(dist * inv_rc) + 1.0f);   // c_ij alone: the record is shared by the message and head passes
            kind = __float_as_int(dv.w);
        }
        int prev = __shfl_up_sync(FULL, row, 1);
        if (lane == 0) prev = -2;                 // a granule is a warp's 32 pairs: its first pair always starts a segment
        const unsigned fm = __ballot_sync(FULL, row != prev);
        // ---- meta slot
        if ((p >> 5) == 1) {                      // poller of role P (warp 1)
            WAITED(tc::mbar_wait(&bar[META_EMPTY + (it & (NM - 1))], ((it / NM) & 1) ^ 1));
            WAITED(tc::mbar_wait(&bar[A1_EMPTY + (it & 1)], ((it >> 1) & 1) ^ 1));
        }
        WAITED(tc::named_bar_sync(NB_P, 128));
        Meta &M = meta_of(S, it);
        if (lane == 0) { M.fmask[2 * (p >> 5)] = fm & 0xFFFFu; M.fmask[2 * (p >> 5) + 1] = fm >> 16; }
        M.w[p] = w; M.jrow[p] = jrow; M.rowk[p] = (row < 0) ? -1 : (row | (kind << 29));
        M.u[0][p] = ux; M.u[1][p] = uy; M.u[2][p] = uz;   // used by the head pass, which re-reads this record
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(&bar[META_FULL + (it & (NM - 1))]);
        // ---- RBF tile -> A1 (bf16, K-major rows of 128 B, 16-byte chunks XOR-swizzled by row & 7)
        unsigned char *A1 = S + OFF_A1 + (it & 1) * 16384 + p * 128;
        const float uc = dist * uc_scale;         // C d / delta
        // Only the basis functions within 8 widths of d are evaluated: three 8-function chunks starting at chunk c0 cover every
        // k with |k - d/delta| <= 8; the others are below exp(-32) = 1.3e-14 of the largest and are stored as zeros.  (Per-thread
        // chunk index, warp-uniform control flow: the pairs of a warp have unrelated distances.)
        const int c0 = min(max((int)floorf((uc * (1.0f / RBF_C) - 8.0f) * 0.125f), 0), 5);
#pragma unroll
        for (int z = 0; z < 5; ++z) {
            const int ch = (z < c0) ? z : z + 3;
            *(uint4 *)(A1 + ((ch ^ (p & 7)) << 4)) = make_uint4(0u, 0u, 0u, 0u);
        }
#pragma unroll
        for (int c3 = 0; c3 < 3; ++c3) {
            const int ch = c0 + c3;
            const float ub = uc - (RBF_C * 8.0f) * (float)ch;
            float g[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const float t = ub - RBF_C * (float)e;
                g[e] = ex2_approx(-t * t);
            }
            *(uint4 *)(A1 + ((ch ^ (p & 7)) << 4)) =
                make_uint4(tc::pack_bf16(g[0], g[1]), tc::pack_bf16(g[2], g[3]), tc::pack_bf16(g[4], g[5]), tc::pack_bf16(g[6], g[7]));
        }
        tc::fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(&bar[A1_FULL + (it & 1)]);
    }
    STATS_END("P")
}

// ---- role H: h1 = SiLU(2 (D1 + b_e1/2)) -> A2.  Thread p owns TMEM lane p (pair p) and all 128 columns.
__device__ __forceinline__ void role_H(const PairArgs &a, unsigned char *S, uint64_t *bar, uint32_t tmem, int n_my, int p, int lane)
{
    STATS_BEGIN
    const uint32_t lane_field = (uint32_t)(p & ~31) << 16;
    for (int it = 0; it < n_my; ++it) {
        const int s = it & 1, ph = (it >> 1) & 1;
        if ((p >> 5) == 2) {                      // poller of role H (warp 6)
            WAITED(tc::mbar_wait(&bar[A2_EMPTY + s], ph ^ 1));
            WAITED(tc::mbar_wait(&bar[D1_FULL + s], ph));
        }
        WAITED(tc::named_bar_sync(NB_H, 128));
        tc::tc_fence_after_sync();
        unsigned char *rowp = S + OFF_A2 + s * 32768 + p * 128;
        const uint32_t td1 = tmem + s * 128 + lane_field;
#pragma unroll
        for (int c2 = 0; c2 < 4; ++c2) {
            uint32_t r0[16], r1[16];
            tc::tmem_ld16_nowait(td1 + c2 * 32, r0);
            tc::tmem_ld16_nowait(td1 + c2 * 32 + 16, r1);
            tc::tmem_ld_wait();
#pragma unroll
            for (int hh = 0; hh < 2; ++hh) {
                const int cc = c2 * 2 + hh;
                uint32_t pk[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int col = cc * 16 + 2 * e;
                    const float h0 = __uint_as_float(hh ? r1[2 * e] : r0[2 * e]) + a.b1h[col];
                    const float h1 = __uint_as_float(hh ? r1[2 * e + 1] : r0[2 * e + 1]) + a.b1h[col + 1];
                    pk[e] = tc::pack_bf16(fmaf(h0, tc::tanh_approx(h0), h0), fmaf(h1, tc::tanh_approx(h1), h1));
                }
                unsigned char *kb = rowp + (cc >> 2) * 16384;
                const int ch0 = (cc & 3) * 2;
                *(uint4 *)(kb + ((ch0 ^ (p & 7)) << 4)) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
                *(uint4 *)(kb + (((ch0 + 1) ^ (p & 7)) << 4)) = make_uint4(pk[4], pk[5], pk[6], pk[7]);
            }
        }
        tc::tc_fence_before_sync();
        tc::fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) { tc::mbar_arrive(&bar[D1_EMPTY + s]); tc::mbar_arrive(&bar[A2_FULL + s]); }
    }
    STATS_END("H")
}

// UMMA shared-memory descriptor, MN-major operand (the contraction index is the shared-memory row), 128-byte swizzle:
// LBO = bytes between 64-element atoms along M/N, SBO = bytes between 8-row groups along K
__device__ __forceinline__ uint64_t make_desc_mn_sw128(uint32_t addr, uint32_t lbo, uint32_t sbo)
{
    return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)((lbo >> 4) & 0x3FFF) << 16) | ((uint64_t)((sbo >> 4) & 0x3FFF) << 32) |
           ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}

// ---- role E, message pass: m_i = agg_norm sum_j c_ij (e0_ij + E_i + E_j) (.) x_j  (S:G3, G5).
// D2 is TRANSPOSED (TMEM lane = channel c, column = pair): the thread walks the 32 pairs of its quarter tile in CSR
// order.  m_i = sum_j c_ij (e0 x_j + y_j) + (b + E_i) sum_j c_ij x_j with y_j = E_j x_j formed once per atom by the node kernel,
// so the two private running sums do not depend on the row and a row boundary only cuts them.  The gathered word carries
// x_j in its low half and IS y_j when read as an fp32 (tc::pack_x_y): per (pair, channel) one shared-memory load, one shift
// and three FMAs.  Lanes = consecutive channels: conflict-free.  E_i comes from the fp32 master (tile-blocked, gfn_node_tc.cu).
// Code is kept small on purpose (five roles share the instruction cache).
struct MsgState {
    int cur, kind;               // current row (-1 none), its segment kind
    float s1, s2, ei;            // running sums; E_i of the row (in flight until the flush)
};

__device__ __forceinline__ void msg_flush(const PairArgs &a, const MsgState &st, int64_t gidx, int c, float b2c)
{
    if (st.cur >= 0) {
        float *dst = (st.kind == 0) ? a.m_out + (size_t)st.cur * H + c : a.carry_m + (size_t)(gidx * 2 + (st.kind - 1)) * H + c;
        *dst = a.wscale * fmaf(b2c + st.ei, st.s2, st.s1);     // wscale = agg_norm
    }
}

// b + E_i of the row that starts: prefetched at the previous boundary (CSR rows are consecutive), else loaded now
__device__ __forceinline__ size_t e_master_off(int row, int c) { return ((size_t)(row >> 7) * (H / 4) + (c >> 2)) * (128 * 4) + (size_t)(row & 127) * 4 + (c & 3); }
// E_i of the row that starts.  The load is only issued here; its value is first used when the segment is flushed, so its
// latency (the fp32 master is not kept in L2 by the gathers the way XE is) hides behind the segment's pairs.
template <bool FIRST>
__device__ __forceinline__ void msg_row_bias(const float *__restrict__ Em, MsgState &st, int c)
{
    st.ei = FIRST ? 0.f : __ldg(Em + e_master_off(st.cur, c));
}

// FIRST: the first message pass of an evaluation is layer 0, where E = 0 for every atom (a4): e_ij = e0_ij + b, so the E_j unpack
// and add, and the E_i loads, are left out (adding the zeros would give the same bits).
template <bool FIRST>
__device__ __forceinline__ void role_E_msg(const PairArgs &a, unsigned char *S, uint64_t *bar, uint32_t tmem, int n_my, int c,
                                           int qt, int lane, bool poller)
{
    STATS_BEGIN
    const float b2c = ((const float *)(S + OFF_BIAS))[H + c];
    const uint32_t lane_field = (uint32_t)(c & ~31) << 16;
    const int64_t stride = (int64_t)gridDim.x * TP;
    int64_t tile0 = (int64_t)blockIdx.x * TP;
    MsgState st;
    st.cur = -1; st.kind = 0; st.s1 = st.s2 = st.ei = 0.f;
    for (int it = 0; it < n_my; ++it, tile0 += stride) {
        const Meta &M = meta_of(S, it);
        const int64_t gidx = (tile0 >> 5) + qt;
        const uint32_t td2 = tmem + 256 + (it & 1) * 128 + lane_field;
        st.s1 = 0.f; st.s2 = 0.f;
#pragma unroll
        for (int cc = 0; cc < 2; ++cc) {
            const int q0 = qt * 32 + cc * 16, slot = qt * 2 + cc;   // ring slot = 16 pairs
            if (poller) {
                if (cc == 0) {
                    WAITED(tc::mbar_wait(&bar[META_FULL + (it & (NM - 1))], (it / NM) & 1));
                    WAITED(tc::mbar_wait(&bar[D2_FULL + (it & 1)], (it >> 1) & 1));
                }
                WAITED(tc::mbar_wait(&bar[XE_FULL + slot], it & 1));   // gathered rows of this slot have landed
            }
            WAITED(tc::named_bar_sync(NB_E + qt, 128));
            if (cc == 0) {
                tc::tc_fence_after_sync();
                // the quarter tile is one granule: its first pair always starts a segment
                const int rk = M.rowk[qt * 32];
                st.cur = (rk < 0) ? -1 : (rk & 0x1FFFFFFF);
                st.kind = (rk < 0) ? 0 : (rk >> 29);
                if (st.cur >= 0) msg_row_bias<FIRST>(a.Emaster, st, c);
            }
            float v[16];
            tc::tmem_ld16(td2 + q0, v);
            if (cc == 1) {                       // accumulator drained: hand D2 back to the MMA warp
                tc::tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) tc::mbar_arrive(&bar[D2_EMPTY + (it & 1)]);
            }
            const uint32_t *xr = (const uint32_t *)(S + OFF_RING + slot * 8192) + c;
            // v <- e0 x_j + y_j, xv <- x_j; the cutoff weights c_ij stay in shared memory and enter in the sums (two FMAs per term)
            float xv[16];
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                const uint32_t xe = xr[e * H];
                xv[e] = tc::bf16lo_to_f32(xe);
                v[e] = FIRST ? v[e] * xv[e] : fmaf(v[e], xv[e], __uint_as_float(xe));
            }
            const float *wq = &M.w[q0];
            unsigned mask = M.fmask[qt * 2 + cc];
            if (cc == 0) mask &= ~1u;            // handled above
            if (mask == 0u) {
#pragma unroll
                for (int e = 0; e < 16; ++e) { const float w = wq[e]; st.s1 = fmaf(w, v[e], st.s1); st.s2 = fmaf(w, xv[e], st.s2); }
            } else if ((mask & (mask - 1)) == 0u) {
                // exactly one row boundary in the chunk (the usual case: rows are longer than 16 pairs): the pairs
                // before it close the running sums, the pairs from it on open the next row's (warp-uniform predicates)
                const int hi = __ffs(mask) - 1;
                float t1 = 0.f, t2 = 0.f;
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    const float w = wq[e];
                    if (e < hi) { st.s1 = fmaf(w, v[e], st.s1); st.s2 = fmaf(w, xv[e], st.s2); }
                    else        { t1 = fmaf(w, v[e], t1); t2 = fmaf(w, xv[e], t2); }
                }
                msg_flush(a, st, gidx, c, b2c);
                const int rk = M.rowk[q0 + hi];
                st.cur = (rk < 0) ? -1 : (rk & 0x1FFFFFFF);
                st.kind = (rk < 0) ? 0 : (rk >> 29);
                st.s1 = t1; st.s2 = t2;
                if (st.cur >= 0) msg_row_bias<FIRST>(a.Emaster, st, c);
            } else {
                int lo = 0;
#pragma unroll 1
                while (true) {                   // warp-uniform: segments [lo, hi) between row boundaries
                    const int hi = mask ? (__ffs(mask) - 1) : 16;
#pragma unroll
                    for (int e = 0; e < 16; ++e)
                        if (e >= lo && e < hi) { const float w = wq[e]; st.s1 = fmaf(w, v[e], st.s1); st.s2 = fmaf(w, xv[e], st.s2); }
                    if (!mask) break;
                    mask &= mask - 1;
                    lo = hi;
                    msg_flush(a, st, gidx, c, b2c);   // a new row segment starts at pair q0 + hi
                    const int rk = M.rowk[q0 + hi];
                    st.cur = (rk < 0) ? -1 : (rk & 0x1FFFFFFF);
                    st.kind = (rk < 0) ? 0 : (rk >> 29);
                    st.s1 = 0.f; st.s2 = 0.f;
                    if (st.cur >= 0) msg_row_bias<FIRST>(a.Emaster, st, c);
                }
            }
            if (it + 1 < n_my) tc::named_bar_arrive(NB_SLOT + slot, 160);   // slot consumed: its refill overlaps the other chunk
        }
        msg_flush(a, st, gidx, c, b2c);
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(&bar[META_EMPTY + (it & (NM - 1))]);
    }
    STATS_END("E")
}

// ---- role E, force head: s_ij = w_f2 . SiLU(W_fe h1 + b_fe + G_i + G_j) + b_f2,  F_i = sum_j c_ij s_ij u_ij  (S:G4).
// Everything is carried as h = t/2.  Per-thread term for channel c, then a fixed-tree transposing reduction over the
// 32 lanes and the 4 lane quadrants; pair-level segmented warp scan over 32-pair granules.
__device__ __forceinline__ void role_E_head(const PairArgs &a, unsigned char *S, uint64_t *bar, uint32_t tmem, int n_my, int c,
                                            int qt, int lane, int e_tid, bool poller)
{
    STATS_BEGIN
    const float b2c = 0.5f * ((const float *)(S + OFF_BIAS))[H + c];
    const float wc = ((const float *)(S + OFF_BIAS))[2 * H + c];
    const float *__restrict__ Gf = (const float *)a.gsrc;
    float *s4 = (float *)(S + OFF_S4);           // [4][TP]
    const int quarter = c >> 5;
    const uint32_t lane_field = (uint32_t)(c & ~31) << 16;
    const int64_t stride = (int64_t)gridDim.x * TP;
    int64_t tile0 = (int64_t)blockIdx.x * TP;
    int nx_row = -1;
    float nx_val = 0.f;
    for (int it = 0; it < n_my; ++it, tile0 += stride) {
        const Meta &M = meta_of(S, it);
        const uint32_t td2 = tmem + 256 + (it & 1) * 128 + lane_field;
        float be = 0.f;
        int cur_row = -2;
#pragma unroll 1
        for (int cc = 0; cc < 2; ++cc) {
            const int q0 = qt * 32 + cc * 16, slot = qt * 2 + cc;   // ring slot = 16 pairs
            if (poller) {
                if (cc == 0) {
                    WAITED(tc::mbar_wait(&bar[META_FULL + (it & (NM - 1))], (it / NM) & 1));
                    WAITED(tc::mbar_wait(&bar[D2_FULL + (it & 1)], (it >> 1) & 1));
                }
                WAITED(tc::mbar_wait(&bar[XE_FULL + slot], it & 1));
            }
            WAITED(tc::named_bar_sync(NB_E + qt, 128));
            if (cc == 0) tc::tc_fence_after_sync();
            float v[16];
            tc::tmem_ld16(td2 + q0, v);
            if (cc == 1) {
                tc::tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) tc::mbar_arrive(&bar[D2_EMPTY + (it & 1)]);
            }
            const float *gr = (const float *)(S + OFF_RING + slot * 8192) + c;
            float gj[16];
#pragma unroll
            for (int e = 0; e < 16; ++e) gj[e] = gr[e * H];
            unsigned mask = M.fmask[qt * 2 + cc];
            if ((mask & 1u) && cc > 0) {         // granule start forced by P: a boundary for G_i only if the row changes
                const int rk = M.rowk[q0];
                if (((rk < 0) ? -1 : (rk & 0x1FFFFFFF)) == cur_row) mask &= ~1u;
            }
            if (mask == 0u) {
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    const float h = fmaf(0.5f, gj[e], v[e] + be);
                    v[e] = wc * fmaf(h, tc::tanh_approx(h), h);
                }
            } else {
                int lo = 0;
#pragma unroll 1
                while (true) {                   // warp-uniform: segments [lo, hi) between row boundaries
                    const int hi = mask ? (__ffs(mask) - 1) : 16;
#pragma unroll
                    for (int e = 0; e < 16; ++e)
                        if (e >= lo && e < hi) {
                            const float h = fmaf(0.5f, gj[e], v[e] + be);
                            v[e] = wc * fmaf(h, tc::tanh_approx(h), h);
                        }
                    if (!mask) break;
                    mask &= mask - 1;
                    lo = hi;
                    const int rk = M.rowk[q0 + hi];
                    const int r = (rk < 0) ? -1 : (rk & 0x1FFFFFFF);
                    cur_row = r;
                    if (r >= 0) {
                        const float raw = (r == nx_row) ? nx_val : __ldg(Gf + (size_t)r * H + c);
                        be = b2c + 0.5f * raw;
                        nx_row = (r + 1 < a.rows) ? r + 1 : r;
                        nx_val = __ldg(Gf + (size_t)nx_row * H + c);
                    }
                }
            }
            if (it + 1 < n_my) tc::named_bar_arrive(NB_SLOT + slot, 160);
            // transposing reduction over the 32 lanes (channels of this quadrant): 16 pairs -> lanes
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const float send = (lane & 16) ? v[i] : v[i + 8], keep = (lane & 16) ? v[i + 8] : v[i];
                v[i] = keep + __shfl_xor_sync(FULL, send, 16);
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float send = (lane & 8) ? v[i] : v[i + 4], keep = (lane & 8) ? v[i + 4] : v[i];
                v[i] = keep + __shfl_xor_sync(FULL, send, 8);
            }
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const float send = (lane & 4) ? v[i] : v[i + 2], keep = (lane & 4) ? v[i + 2] : v[i];
                v[i] = keep + __shfl_xor_sync(FULL, send, 4);
            }
            {
                const float send = (lane & 2) ? v[0] : v[1], keep = (lane & 2) ? v[1] : v[0];
                v[0] = keep + __shfl_xor_sync(FULL, send, 2);
            }
            v[0] += __shfl_xor_sync(FULL, v[0], 1);
            // lane bits (4,3,2,1) select pair e = 8 b4 + 4 b3 + 2 b2 + b1
            if ((lane & 1) == 0)
                s4[quarter * TP + q0 + ((lane >> 4) & 1) * 8 + ((lane >> 3) & 1) * 4 + ((lane >> 2) & 1) * 2 + ((lane >> 1) & 1)] = v[0];
        }
        WAITED(tc::named_bar_sync(NB_S4, 512));          // s4 of this tile complete
        if (e_tid < TP) {
            const int p = e_tid;
            const int rk = M.rowk[p];
            const int key = (rk < 0) ? -1 : (rk & 0x1FFFFFFF);
            const float f = M.w[p] * (((s4[p] + s4[TP + p]) + (s4[2 * TP + p] + s4[3 * TP + p])) + a.bf2);
            float fv[3] = {f * M.u[0][p], f * M.u[1][p], f * M.u[2][p]};
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int ko = __shfl_up_sync(FULL, key, o);
#pragma unroll
                for (int ax = 0; ax < 3; ++ax) {
                    const float vo = __shfl_up_sync(FULL, fv[ax], o);
                    if (lane >= o && ko == key) fv[ax] += vo;
                }
            }
            const int knext = __shfl_down_sync(FULL, key, 1);
            if (key >= 0 && (lane == 31 || knext != key)) {
                const int kind = rk >> 29;
                const int64_t gidx = (tile0 + (p & ~31)) >> 5;
                float *dst = (kind == 0) ? a.Fraw + (size_t)key * 4 : a.carry_f + (size_t)(gidx * 2 + (kind - 1)) * 4;
                dst[0] = fv[0]; dst[1] = fv[1]; dst[2] = fv[2];
            }
        }
        WAITED(tc::named_bar_sync(NB_S4, 512));          // s4 free for the next tile
        if (lane == 0) tc::mbar_arrive(&bar[META_EMPTY + (it & (NM - 1))]);
    }
    STATS_END("Eh")
}

// ---- role E, force head with the channel reduction on the tensor core (HEAD, MODE 1):
// act[p][c] = SiLU(W_fe h1 + b_fe + G_i + G_j)[c] is written as a bf16 MN-major operand (A3: row = channel, pairs contiguous); the MMA warp forms
// D3[p][.] = act[p][:] . w_f2 (128x16x128), and role F turns s_p into forces.  No shuffles, no CTA-wide barrier.
__device__ __forceinline__ void role_E_head_tc(const PairArgs &a, unsigned char *S, uint64_t *bar, uint32_t tmem, int n_my, int c,
                                               int qt, int lane, bool poller)
{
    STATS_BEGIN
    const float b2c = 0.5f * ((const float *)(S + OFF_BIAS))[H + c];
    const float *__restrict__ Gf = (const float *)a.gsrc;
    const uint32_t lane_field = (uint32_t)(c & ~31) << 16;
    const int a3_off = (c >> 3) * 1024 + (c & 7) * 128;      // A3 is MN-major (pairs contiguous): row = channel, 8-channel groups 1 KB apart
    int nx_row = -1;
    float nx_val = 0.f;
    for (int it = 0; it < n_my; ++it) {
        const Meta &M = meta_of(S, it);
        const int s3 = it & 1;
        unsigned char *A3 = S + (s3 ? OFF_A1 : OFF_A2 + 32768) + a3_off;
        const uint32_t td2 = tmem + 256 + (it & 1) * 128 + lane_field;
        float be = 0.f;
        int cur_row = -2;
#pragma unroll
        for (int cc = 0; cc < 2; ++cc) {
            const int q0 = qt * 32 + cc * 16, slot = qt * 2 + cc;
            if (poller) {
                if (cc == 0) {
                    WAITED(tc::mbar_wait(&bar[META_FULL + (it & (NM - 1))], (it / NM) & 1));
                    WAITED(tc::mbar_wait(&bar[D2_FULL + (it & 1)], (it >> 1) & 1));
                    WAITED(tc::mbar_wait(&bar[A3_EMPTY + s3], ((it >> 1) & 1) ^ 1));
                }
                WAITED(tc::mbar_wait(&bar[XE_FULL + slot], it & 1));
            }
            WAITED(tc::named_bar_sync(NB_E + qt, 128));
            if (cc == 0) tc::tc_fence_after_sync();
            float v[16];
            tc::tmem_ld16(td2 + q0, v);
            if (cc == 1) {
                tc::tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) tc::mbar_arrive(&bar[D2_EMPTY + (it & 1)]);
            }
            const float *gr = (const float *)(S + OFF_RING + slot * 8192) + c;
            float gj[16];
#pragma unroll
            for (int e = 0; e < 16; ++e) gj[e] = gr[e * H];
            unsigned mask = M.fmask[qt * 2 + cc];
            if (mask & 1u) {                     // granule start forced by P: a boundary for G_i only if the row changes
                const int rk = M.rowk[q0];
                const int r = (rk < 0) ? -1 : (rk & 0x1FFFFFFF);
                if (r != cur_row) {              // handled here, so that the chunk takes the branch-free path
                    cur_row = r;
                    if (r >= 0) {
                        const float raw = (r == nx_row) ? nx_val : __ldg(Gf + (size_t)r * H + c);
                        be = b2c + 0.5f * raw;
                        nx_row = (r + 1 < a.rows) ? r + 1 : r;
                        nx_val = __ldg(Gf + (size_t)nx_row * H + c);
                    }
                }
                mask &= ~1u;
            }
            if (mask == 0u) {
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    const float h = fmaf(0.5f, gj[e], v[e] + be);
                    v[e] = fmaf(h, tc::tanh_approx(h), h);
                }
            } else if ((mask & (mask - 1)) == 0u) {
                // exactly one row boundary in the chunk (the usual case): pairs before it take the old row's bias,
                // pairs from it on the new row's (warp-uniform select)
                const int hi = __ffs(mask) - 1;
                const float be0 = be;
                const int rk = M.rowk[q0 + hi];
                const int r = (rk < 0) ? -1 : (rk & 0x1FFFFFFF);
                cur_row = r;
                if (r >= 0) {
                    const float raw = (r == nx_row) ? nx_val : __ldg(Gf + (size_t)r * H + c);
                    be = b2c + 0.5f * raw;
                    nx_row = (r + 1 < a.rows) ? r + 1 : r;
                    nx_val = __ldg(Gf + (size_t)nx_row * H + c);
                }
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    const float h = fmaf(0.5f, gj[e], v[e] + ((e < hi) ? be0 : be));
                    v[e] = fmaf(h, tc::tanh_approx(h), h);
                }
            } else {
                int lo = 0;
#pragma unroll 1
                while (true) {                   // warp-uniform: segments [lo, hi) between row boundaries
                    const int hi = mask ? (__ffs(mask) - 1) : 16;
#pragma unroll
                    for (int e = 0; e < 16; ++e)
                        if (e >= lo && e < hi) {
                            const float h = fmaf(0.5f, gj[e], v[e] + be);
                            v[e] = fmaf(h, tc::tanh_approx(h), h);
                        }
                    if (!mask) break;
                    mask &= mask - 1;
                    lo = hi;
                    const int rk = M.rowk[q0 + hi];
                    const int r = (rk < 0) ? -1 : (rk & 0x1FFFFFFF);
                    cur_row = r;
                    if (r >= 0) {
                        const float raw = (r == nx_row) ? nx_val : __ldg(Gf + (size_t)r * H + c);
                        be = b2c + 0.5f * raw;
                        nx_row = (r + 1 < a.rows) ? r + 1 : r;
                        nx_val = __ldg(Gf + (size_t)nx_row * H + c);
                    }
                }
            }
            if (it + 1 < n_my) tc::named_bar_arrive(NB_SLOT + slot, 160);
            // act -> A3: the thread's 16 pairs are two 16-byte chunks of its channel's row (64-pair atoms 16 KB apart,
            // chunks XOR-swizzled by channel & 7): two 128-bit stores instead of sixteen 16-bit ones
            {
                unsigned char *row = A3 + (q0 >> 6) * 16384;
                const int ch0 = (q0 & 63) >> 3;
                // fp16, not bf16: the readout sums 128 signed terms w_f2[c] act[c] that cancel, and the emulation
                // (tests/test_bf16_emulation.py) shows a bf16 operand here alone costs 0.4-0.5 % rms of |F|; SiLU output is far inside
                // the fp16 range (a value beyond it saturates to inf and trips the non-finite force check)
                *(uint4 *)(row + ((ch0 ^ (c & 7)) << 4)) =
                    make_uint4(tc::pack_f16(v[0], v[1]), tc::pack_f16(v[2], v[3]), tc::pack_f16(v[4], v[5]), tc::pack_f16(v[6], v[7]));
                *(uint4 *)(row + (((ch0 + 1) ^ (c & 7)) << 4)) =
                    make_uint4(tc::pack_f16(v[8], v[9]), tc::pack_f16(v[10], v[11]), tc::pack_f16(v[12], v[13]), tc::pack_f16(v[14], v[15]));
            }
        }
        tc::fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) { tc::mbar_arrive(&bar[A3_FULL + s3]); tc::mbar_arrive(&bar[META_EMPTY + (it & (NM - 1))]); }
    }
    STATS_END("Et")
}

// ---- role F (HEAD, MODE 1; the four warps that are role H in the first pass): s_p from D3 -> F_i = sum_j c_ij s_ij u_ij by a
// segmented warp scan over 32-pair granules (S:G4).  Thread p owns pair p = TMEM lane p.
__device__ __forceinline__ void role_F(const PairArgs &a, unsigned char *S, uint64_t *bar, uint32_t tmem, int n_my, int p, int lane)
{
    STATS_BEGIN
    const uint32_t lane_field = (uint32_t)(p & ~31) << 16;
    const int64_t stride = (int64_t)gridDim.x * TP;
    int64_t tile0 = (int64_t)blockIdx.x * TP;
    for (int it = 0; it < n_my; ++it, tile0 += stride) {
        const Meta &M = meta_of(S, it);
        const int s = it & 1;
        if ((p >> 5) == 2) {
            WAITED(tc::mbar_wait(&bar[META_FULL + (it & (NM - 1))], (it / NM) & 1));
            WAITED(tc::mbar_wait(&bar[D3_FULL + s], (it >> 1) & 1));
        }
        WAITED(tc::named_bar_sync(NB_H, 128));
        tc::tc_fence_after_sync();
        const float sp = tc::tmem_ld1(tmem + s * 32 + lane_field);
        tc::tc_fence_before_sync();
        const int rk = M.rowk[p];
        const int key = (rk < 0) ? -1 : (rk & 0x1FFFFFFF);
        const float f = M.w[p] * (sp + a.bf2);
        float fv[3] = {f * M.u[0][p], f * M.u[1][p], f * M.u[2][p]};
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int ko = __shfl_up_sync(FULL, key, o);
#pragma unroll
            for (int ax = 0; ax < 3; ++ax) {
                const float vo = __shfl_up_sync(FULL, fv[ax], o);
                if (lane >= o && ko == key) fv[ax] += vo;
            }
        }
        const int knext = __shfl_down_sync(FULL, key, 1);
        if (key >= 0 && (lane == 31 || knext != key)) {
            const int kind = rk >> 29;
            const int64_t gidx = (tile0 + (p & ~31)) >> 5;
            float *dst = (kind == 0) ? a.Fraw + (size_t)key * 4 : a.carry_f + (size_t)(gidx * 2 + (kind - 1)) * 4;
            dst[0] = fv[0]; dst[1] = fv[1]; dst[2] = fv[2];
        }
        __syncwarp();
        if (lane == 0) { tc::mbar_arrive(&bar[D3_EMPTY + s]); tc::mbar_arrive(&bar[META_EMPTY + (it & (NM - 1))]); }
    }
    STATS_END("F")
}

// ---- role MMA: one elected lane issues both products; completion is committed to the consumers' mbarriers
template <bool HEAD, int MODE>
__device__ __forceinline__ void role_MMA(const PairArgs &a, unsigned char *S, uint64_t *bar, uint32_t tmem, int n_my, int lane)
{
    STATS_BEGIN
    constexpr bool TCH = HEAD && MODE == 1;      // head with the channel reduction on the tensor core
    constexpr int NA2 = TCH ? 1 : 2;             // A2 stages (the second stage's space is an A3 stage there)
    const uint32_t idesc = tc::make_idesc_bf16(TP, H), idesc16 = tc::make_idesc_f16(TP, 16);   // readout product: fp16 operands
    const uint32_t sW1 = tc::smem_u32(S + OFF_W1), sW2 = tc::smem_u32(S + OFF_W2);
    const uint32_t sA1 = tc::smem_u32(S + OFF_A1), sA2 = tc::smem_u32(S + OFF_A2);
    tc::mbar_wait(&bar[W_FULL], 0);
    for (int k = 0; k <= n_my + (TCH ? 1 : 0); ++k) {
        if (MODE == 0 && k < n_my) {             // D1[s] = G (W_e1/2)^T   (4 x UMMA 128x128x16)
            const int s = k & 1, ph = (k >> 1) & 1;
            WAITED(LAZY_WAIT(&bar[D1_EMPTY + s], ph ^ 1));
            WAITED(LAZY_WAIT(&bar[A1_FULL + s], ph));
            tc::tc_fence_after_sync();
            if (lane == 0) {
#pragma unroll
                for (int kk = 0; kk < K / 16; ++kk)
                    tc::mma_bf16_ss(tmem + s * 128, tc::make_desc_sw128(sA1 + s * 16384 + kk * 32),
                                    tc::make_desc_sw128(sW1 + kk * 32), idesc, kk > 0);
                tc::mma_commit(&bar[D1_FULL + s]);
                tc::mma_commit(&bar[A1_EMPTY + s]);
            }
            __syncwarp();
        }
        if (k >= 1 && k <= n_my) {               // D2[s]^T = W2 h1^T   (8 x UMMA; M = channels, N = pairs)
            const int j = k - 1, s = j & 1, ph = (j >> 1) & 1, sa = j % NA2, pha = (j / NA2) & 1;
            WAITED(LAZY_WAIT(&bar[D2_EMPTY + s], ph ^ 1));
            WAITED(LAZY_WAIT(&bar[A2_FULL + sa], pha));
            tc::tc_fence_after_sync();
            if (lane == 0) {
#pragma unroll
                for (int kk = 0; kk < H / 16; ++kk) {
                    const uint32_t off = (kk >> 2) * 16384 + (kk & 3) * 32;
                    tc::mma_bf16_ss(tmem + 256 + s * 128, tc::make_desc_sw128(sW2 + off),
                                    tc::make_desc_sw128(sA2 + sa * 32768 + off), idesc, kk > 0);
                }
                tc::mma_commit(&bar[D2_FULL + s]);
                tc::mma_commit(&bar[A2_EMPTY + sa]);
            }
            __syncwarp();
        }
        if (TCH && k >= 2) {                     // D3[s][p][0..15] = act[p][:] . w_f2   (8 x UMMA 128x16x16; M = pairs)
            const int i = k - 2, s = i & 1, ph = (i >> 1) & 1;
            WAITED(LAZY_WAIT(&bar[D3_EMPTY + s], ph ^ 1));
            WAITED(LAZY_WAIT(&bar[A3_FULL + s], ph));
            tc::tc_fence_after_sync();
            if (lane == 0) {
                const uint32_t sA3 = s ? sA1 : sA2 + 32768;
#pragma unroll
                for (int kk = 0; kk < H / 16; ++kk)      // A3 MN-major: a K step is two 8-channel groups (2 KB); 64-pair atoms 16 KB apart
                    tc::mma_bf16_ss(tmem + s * 32, make_desc_mn_sw128(sA3 + kk * 2048, 16384, 1024),
                                    tc::make_desc_sw128(sW1 + (kk >> 2) * 2048 + (kk & 3) * 32), idesc16 | (1u << 15), kk > 0);
                tc::mma_commit(&bar[D3_FULL + s]);
                tc::mma_commit(&bar[A3_EMPTY + s]);
            }
            __syncwarp();
        }
    }
    STATS_END("MMA")
}

// ---- role G: gathered rows (512 B each) -> ring slots by TMA bulk copies.  Warp g feeds the two 16-pair slots of
// quarter tile g, one copy per lane (the copy instruction issues from the uniform datapath, one lane at a time).  A slot
// is refilled as soon as the E warps release it, i.e. while they work on the quarter's other slot.
__device__ __forceinline__ void role_G(const PairArgs &a, unsigned char *S, uint64_t *bar, int n_my, int qt, int lane)
{
    STATS_BEGIN
    const int slot = qt * 2 + (lane >> 4);       // lanes 0-15 feed slot 2 qt, lanes 16-31 slot 2 qt + 1
    unsigned char *dst = S + OFF_RING + slot * 8192 + (lane & 15) * 512;
    for (int it = 0; it < n_my; ++it) {
        const Meta &M = meta_of(S, it);
        WAITED(tc::mbar_wait(&bar[META_FULL + (it & (NM - 1))], (it / NM) & 1));
        const int jrow = M.jrow[qt * 32 + lane];
        const int j1 = __shfl_down_sync(FULL, jrow, 1), j2 = __shfl_down_sync(FULL, jrow, 2), j3 = __shfl_down_sync(FULL, jrow, 3);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            if (it > 0) {                                    // the consumers have read the slot
                WAITED(tc::named_bar_sync(NB_SLOT + qt * 2 + h, 160));   // the 128 consumers + this warp
            }
            // four gathered rows (4 x 512 B, consecutive in the slot) per copy: lanes 0, 4, 8, 12 of the half warp issue.  The
            // copies are on the consumers' critical path (slot read -> slot refilled); the barrier's arrival with the byte count is
            // not and follows them (the phase cannot complete before it, whatever has landed by then).
            if ((lane >> 4) == h && (lane & 3) == 0) tc::tma_gather4(dst, &a.gmap, jrow, j1, j2, j3, &bar[XE_FULL + slot]);
            if (lane == 16 * h) tc::mbar_arrive_expect_tx(&bar[XE_FULL + qt * 2 + h], 8192);
        }
    }
    STATS_END("G")
}

// ---- role S (MODE 0): stream every tile's h1 operand image and meta record to HBM for the later passes
__device__ __forceinline__ void role_S(const PairArgs &a, unsigned char *S, uint64_t *bar, int n_my, int lane)
{
    STATS_BEGIN
    for (int it = 0; it < n_my; ++it) {
        const int s = it & 1;
        const int64_t tile = (int64_t)blockIdx.x + (int64_t)it * gridDim.x;
        WAITED(tc::mbar_wait(&bar[META_FULL + (it & (NM - 1))], (it / NM) & 1));
        WAITED(LAZY_WAIT(&bar[A2_FULL + s], (it >> 1) & 1));
        if (lane == 0) {
            tc::fence_proxy_async_smem();       // generic-proxy writes of P and H (acquired above) -> async-proxy reads
            tc::bulk_s2g(a.h1_img + tile * 32768, S + OFF_A2 + s * 32768, 32768);
            tc::bulk_s2g(a.meta_img + tile * (int64_t)sizeof(Meta), &meta_of(S, it), (uint32_t)sizeof(Meta));
            tc::bulk_commit();
            tc::bulk_wait_read();               // shared-memory sources read: the buffers may be refilled
            tc::mbar_arrive(&bar[A2_EMPTY + s]);
            tc::mbar_arrive(&bar[META_EMPTY + (it & (NM - 1))]);
        }
        __syncwarp();
    }
    if (lane == 0) tc::bulk_wait_all();         // global writes complete before the kernel ends
    STATS_END("S")
}

// ---- role L (MODE 1): bring the tile's h1 operand image and meta record back (two TMA bulk copies)
template <int NA2>
__device__ __forceinline__ void role_L(const PairArgs &a, unsigned char *S, uint64_t *bar, int n_my, int lane)
{
    STATS_BEGIN
    for (int it = 0; it < n_my; ++it) {
        const int s = it % NA2, m = it & (NM - 1);
        const int64_t tile = (int64_t)blockIdx.x + (int64_t)it * gridDim.x;
        WAITED(tc::mbar_wait(&bar[META_EMPTY + m], ((it / NM) & 1) ^ 1));
        WAITED(tc::mbar_wait(&bar[A2_EMPTY + s], ((it / NA2) & 1) ^ 1));
        if (lane == 0) {
            tc::mbar_arrive_expect_tx(&bar[META_FULL + m], (uint32_t)sizeof(Meta));
            tc::bulk_g2s(&meta_of(S, it), a.meta_img + tile * (int64_t)sizeof(Meta), (uint32_t)sizeof(Meta), &bar[META_FULL + m]);
            tc::mbar_arrive_expect_tx(&bar[A2_FULL + s], 32768);
            tc::bulk_g2s(S + OFF_A2 + s * 32768, a.h1_img + tile * 32768, 32768, &bar[A2_FULL + s]);
        }
        if (a.Emaster != nullptr) {
            // E_i of the tile's rows (role E loads it per row segment) is touched once per pass and does not stay in L2 behind the
            // image stream: this warp, two tiles ahead of role E, pulls the rows' lines into L2 (4 rows x 32 sectors)
            const int64_t p0 = tile * TP;
            const int r0 = __ldg(a.pair_row + p0);
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int r = r0 + k;
                if (r < a.rows) asm volatile("prefetch.global.L2 [%0];" ::"l"(a.Emaster + e_master_off(r, lane * 4)));
            }
        }
        __syncwarp();
    }
    STATS_END("L")
}

template <bool HEAD, int MODE>
__global__ void __launch_bounds__(Warps<HEAD, MODE>::THREADS, 1) pair_pipe_kernel(const __grid_constant__ PairArgs a)
{ pdl_enter();
    using WL = Warps<HEAD, MODE>;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char *S = smem_raw + ((1024u - (tc::smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t *bar = (uint64_t *)(S + OFF_BAR);
    uint32_t *tmem_slot = (uint32_t *)(S + OFF_TMEM);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int64_t n_pairs = a.row_ptr[a.rows];
    const int n_my = n_my_tiles(n_pairs);

    if (tid == 0) {
        for (int s = 0; s < 2; ++s) {
            tc::mbar_init(&bar[A1_FULL + s], 4);  tc::mbar_init(&bar[A1_EMPTY + s], 1);
            tc::mbar_init(&bar[D1_FULL + s], 1);  tc::mbar_init(&bar[D1_EMPTY + s], 4);
            tc::mbar_init(&bar[A3_FULL + s], 16); tc::mbar_init(&bar[A3_EMPTY + s], 1);
            tc::mbar_init(&bar[D3_FULL + s], 1);  tc::mbar_init(&bar[D3_EMPTY + s], 4);
            tc::mbar_init(&bar[A2_FULL + s], MODE == 0 ? 4 : 1);  tc::mbar_init(&bar[A2_EMPTY + s], MODE == 0 ? 2 : 1);
            tc::mbar_init(&bar[D2_FULL + s], 1);  tc::mbar_init(&bar[D2_EMPTY + s], 16);
        }
        for (int s = 0; s < 2 * NSLOT; ++s) { tc::mbar_init(&bar[XE_FULL + s], 1); }
        for (int s = 0; s < NM; ++s) { tc::mbar_init(&bar[META_FULL + s], MODE == 0 ? 4 : 1); tc::mbar_init(&bar[META_EMPTY + s], MODE == 0 ? 17 : (HEAD ? 20 : 16)); }
        tc::mbar_init(&bar[W_FULL], 1);
        tc::fence_mbar_init();
    }
    if (warp == WL::MMA) tc::tmem_alloc(tmem_slot, 512);
    {
        float *sb = (float *)(S + OFF_BIAS);
        for (int i = tid; i < H; i += WL::THREADS) {
            sb[H + i] = a.b2[i];
            sb[2 * H + i] = HEAD ? a.wf2[i] : 0.f;
        }
    }
    tc::tc_fence_before_sync();
    __syncthreads();
    tc::tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot;
    if (tid == WL::G0 * 32) {                        // filter weights: two TMA bulk copies of pre-swizzled bf16 images
        tc::mbar_arrive_expect_tx(&bar[W_FULL], (MODE == 0 ? 16384 : (HEAD ? 4096 : 0)) + 32768);
        if (MODE == 0) tc::bulk_g2s(S + OFF_W1, a.W1img, 16384, &bar[W_FULL]);
        else if (HEAD) tc::bulk_g2s(S + OFF_W1, a.Wf2img, 4096, &bar[W_FULL]);   // w_f2 operand of the readout product
        tc::bulk_g2s(S + OFF_W2, a.W2img, 32768, &bar[W_FULL]);
    }
    if (MODE == 0) {                               // register re-balancing between warpgroups (aligned groups of 4 warps)
        if (warp < 8) asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        else if (warp < 24) asm volatile("setmaxnreg.inc.sync.aligned.u32 80;");
        else asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
    } else if (HEAD) {                             // 28 warps, 72 at launch: F 56, G and MMA/L 40 -> E 88  (measured: no gain for the
                                                   // later message passes, which run 22 warps at 80 registers)
        if (warp < 16) asm volatile("setmaxnreg.inc.sync.aligned.u32 88;");
        else if (warp < 20) asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        else asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
    }
    if (MODE == 0 && warp < 4) {
        role_P<HEAD>(a, S, bar, n_my, n_pairs, tid, lane);
    } else if (MODE == 0 && warp < 8) {
        role_H(a, S, bar, tmem, n_my, tid - 128, lane);
    } else if (warp >= WL::E0 && warp < WL::E0 + 16) {
        const int we = warp - WL::E0, c = (we & 3) * 32 + lane, qt = we >> 2;
        const bool poller = (we == 1) || (we == 6) || (we == 11) || (we == 12);   // one per quarter, spread over the sub-partitions
        if (HEAD && MODE == 1) role_E_head_tc(a, S, bar, tmem, n_my, c, qt, lane, poller);
        else if (HEAD) role_E_head(a, S, bar, tmem, n_my, c, qt, lane, tid - WL::E0 * 32, poller);
        else role_E_msg<MODE == 0>(a, S, bar, tmem, n_my, c, qt, lane, poller);
    } else if (HEAD && MODE == 1 && warp >= WL::F0 && warp < WL::F0 + 4) {
        role_F(a, S, bar, tmem, n_my, tid - WL::F0 * 32, lane);
    } else if (warp == WL::MMA) {
        role_MMA<HEAD, MODE>(a, S, bar, tmem, n_my, lane);
    } else if (warp >= WL::G0 && warp < WL::G0 + 4) {
        role_G(a, S, bar, n_my, warp - WL::G0, lane);
    } else if (warp == WL::SL) {
        if (MODE == 0) role_S(a, S, bar, n_my, lane);
        else role_L<(HEAD ? 1 : 2)>(a, S, bar, n_my, lane);
    }
    tc::tc_fence_before_sync();
    __syncthreads();
    if (warp == WL::MMA) tc::tmem_dealloc(tmem, 512);
}


int launch_pair_pipe(pimd_ctx *c, bool head, bool first)
{
    PairArgs a;
    a.N = c->N;
    a.r_cut = c->net.r_cut; a.wscale = head ? 1.0f : c->net.agg_norm;
    a.row_ptr = c->nl.row_ptr; a.col = c->nl.col; a.pair_row = c->nl.pair_row; a.dvec = c->nl.dvec; a.rows = c->rows;
    a.W1img = c->wimg_e1; a.W2img = head ? c->wimg_fe : c->wimg_e2; a.Wf2img = c->wimg_wf2;
    for (int k = 0; k < H; ++k) a.b1h[k] = c->h_be1_half[k];
    a.b2 = head ? c->net.bfe : c->net.be2;
    a.gsrc = head ? (const void *)c->Gfeat : (const void *)c->XE;
    a.Emaster = head ? nullptr : c->Efeat;
    a.wf2 = c->net.wf2; a.bf2 = c->net.bf2;
    a.m_out = c->mfeat; a.carry_m = c->carry_m; a.Fraw = c->Fraw; a.carry_f = c->carry_f;
    a.h1_img = c->h1_img; a.meta_img = c->meta_img;
    a.gmap = head ? c->tmap_g : c->tmap_xe;
    const size_t smem = SMEM_BYTES + 1024;
    if (!(c->attr_done & ATTR_PIPE)) {
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(pair_pipe_kernel<false, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(pair_pipe_kernel<false, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(pair_pipe_kernel<true, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(pair_pipe_kernel<true, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        c->attr_done |= ATTR_PIPE;
    }
    if (head) {
        if (first) pimd_launch(pair_pipe_kernel<true, 0>, c->num_sms, Warps<true, 0>::THREADS, smem, c->stream, a);
        else pimd_launch(pair_pipe_kernel<true, 1>, c->num_sms, Warps<true, 1>::THREADS, smem, c->stream, a);
    } else {
        if (first) pimd_launch(pair_pipe_kernel<false, 0>, c->num_sms, Warps<false, 0>::THREADS, smem, c->stream, a);
        else pimd_launch(pair_pipe_kernel<false, 1>, c->num_sms, Warps<false, 1>::THREADS, smem, c->stream, a);
    }
    c->launches++;
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}

}  // namespace gfn_pipe
