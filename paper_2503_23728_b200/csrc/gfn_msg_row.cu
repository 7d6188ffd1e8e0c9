// gfn_msg_row.cu -- message pass of the GFN force net (row a5 of SURVEY 8(a); P:L74 phi_m) with BOTH contractions on
// the 5th-gen tensor cores: the filter MLP per pair slot and the sum over the neighbours of a row.  bf16 operands, fp32
// accumulation in TMEM.  Used when gemm_dtype == 1 and (K, H) == (64, 128)  (BASELINE configs[3..4]).
//
//   m_i[c] = agg sum_j c_ij (e0_ij[c] + b[c] + E_i[c] + E_j[c]) x_j[c],   e0_ij = W_e2 h1_ij,  h1_ij = SiLU(W_e1 g(d_ij) + b_e1)   (S:G2, G3, G5)
// is evaluated with the sum over the neighbours FIRST (exact algebra, no approximation):
//   T_i[c][k] = sum_j x_j[c] (c_ij h1_ij[k])            one 128 x 128 accumulator per row i: contraction over the row's pair slots
//   s_i[c]    = sum_j x_j[c] c_ij ,  t_i[c] = sum_j (E_j x_j)[c] c_ij
//   m_i[c]    = agg ( sum_k W_e2[c][k] T_i[c][k] + (b[c] + E_i[c]) s_i[c] + t_i[c] )
// The neighbour list pads every row to a multiple of 16 pair slots (nlist_kernels.cu, pad16), so a row is a whole number of
// K blocks of 16 slots and nothing in the contraction depends on the data: no masks, no restaging, one accumulator per row.
// Both UMMA operands of the row contraction are MN-major (the pair slot is the K index):
//   A  the gathered rows [x_j | y_j = E_j x_j] (bf16, 512 B per atom): TMA tile::gather4 through a 128-byte-swizzled tensor map
//      writes them straight into the operand layout, four slots per copy and 64-channel plane: no thread ever touches them;
//   B  c_ij h1_ij (bf16) as role H leaves it, plus a third 64-column plane whose first two columns hold c_ij as a bf16 pair
//      hi + lo: columns 128, 129 of the N = 144 product are s_i, and a second product y x [c] (N = 16) gives t_i.
// The filter is evaluated again in every pass (geometry -> Gaussian basis -> W_e1 product -> SiLU): nothing per pair is stored
// between passes, the per-pass HBM traffic is the list and the node arrays only.
//
// One persistent CTA per SM owns a contiguous range of whole rows (nl.part: about equal slot counts) and walks its slots in
// tiles of 128.  Roles (16 warps; mbarriers and named barriers only, no CTA-wide barrier in the loop):
//   P    warps 0-3,  thread = slot : indices, fp64 minimum image -> d, c_ij; K-block row flags; Gaussian basis -> A1 (bf16, K-major)
//   H    warps 4-7,  thread = slot : D1 (TMEM) + b -> SiLU -> x c_ij -> B planes (bf16) + the c_ij columns
//   EPI  warps 8-11, thread = channel c (TMEM lane): row c of W_e2 in 128 registers; per finished row the three terms above -> m_i
//   MMA  warp 12, one thread       : D1 = A1 (W_e1/2)^T per tile; per K block T (+)= X^T B (128 x 144 x 16) and t (+)= Y^T [c] (128 x 16 x 16)
//   G    warps 13 (x planes), 14 (y planes): gather4 copies into a ring of 32-slot stages
// Determinism: every sum has a fixed order (K blocks in list order into one accumulator; fixed-order epilogue): bitwise reproducible.
#include "common.cuh"
#include "tc_ptx.cuh"

namespace gfn_row {

constexpr int TP = 128;      // slots per tile
constexpr int H = 128;       // channels
constexpr int K = 64;        // radial basis functions
constexpr int NM = 4;        // meta ring depth (tiles)
constexpr int SB = 32;       // slots per gather stage (two K blocks)
constexpr int ACC_COLS = 160;                 // T 0-127 | s 128-143 | t 144-159
constexpr int TM_D1 = 0, TM_ACC = 128;        // TMEM columns: D1 (128), two row accumulators (2 x 160)
constexpr int THREADS = 512;
constexpr int W_P = 0, W_H = 4, W_EPI = 8, W_MMA = 12, W_G = 13;

struct Args {
    alignas(64) CUtensorMap gmap;         // XY table [rows][256 bf16] (x | y), box = 64 columns x 1 row, 128-byte swizzle
    int N, periodic;
    double box[3], inv_box[3];
    float r_cut, agg;
    const int *row_ptr, *col, *pair_row, *part;
    int64_t rows;
    const double *q;
    const uint16_t *W1img;                // bf16 UMMA image of 0.5 W_e1 [128][64]
    float b1h[H];                         // b_e1 / 2
    const float *We2T;                    // fp32 [k][c]
    const float *b2;                      // b_e2
    const float *E;                       // fp32 master of the running edge sums, tile-blocked (gfn_node_tc.cu); unused in the first layer
    float *m_out;                         // [rows][H]
};

struct Meta {
    float w[TP];                 // c_ij (0 in padding slots and past the end of the range)
    int jrow[TP];                // global row of atom j (own row in padding slots: any finite row will do)
    unsigned kflag[4];           // per P warp (32 slots = K blocks 2w, 2w+1): bits 0-1 block starts a row, bits 8-9 block ends a row
    unsigned pad_[4];
};
static_assert(sizeof(Meta) % 16 == 0, "Meta alignment");

template <bool FIRST> struct Cfg {
    static constexpr int PLANES = FIRST ? 2 : 4;
    static constexpr int STAGE = PLANES * SB * 128;            // bytes: [plane][32 slots][128 B]
    static constexpr int NG = FIRST ? 1 : 2;                   // gather warps
};

constexpr int OFF_W1 = 0;                          // 16 KB
constexpr int OFF_A1 = OFF_W1 + 16384;             // 16 KB
constexpr int OFF_B = OFF_A1 + 16384;              // 2 stages x 3 planes x 16 KB
constexpr int B_STAGE = 3 * 16384;
constexpr int OFF_RING = OFF_B + 2 * B_STAGE;      // 80 KB: 5 stages of 16 KB, or 10 of 8 KB in the first layer
constexpr int RING_BYTES = 81920;
constexpr int OFF_META = OFF_RING + RING_BYTES;
constexpr int OFF_BAR = OFF_META + NM * (int)sizeof(Meta);
constexpr int N_BAR = 48;
constexpr int OFF_TMEM = OFF_BAR + N_BAR * 8;
constexpr int SMEM_BYTES = OFF_TMEM + 16;
static_assert(SMEM_BYTES + 1024 <= 232448, "shared memory carve exceeds 227 KB");

enum { NB_P = 1, NB_H = 2, NB_EPI = 3 };
enum { A1_FULL = 0, A1_EMPTY = 1, D1_FULL = 2, D1_EMPTY = 3, B_FULL = 4, B_EMPTY = 6, META_FULL = 8, META_EMPTY = 12,
       ACC_FULL = 16, ACC_EMPTY = 18, W_FULL = 20, RING_FULL = 24, RING_EMPTY = 36 };   // RING_*: up to 12 stages

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
constexpr float RBF_C = 0.84932180028801904f;   // sqrt(0.5 log2 e): exp(-t^2/2) = 2^-(C t)^2
constexpr unsigned FULL = 0xffffffffu;

__device__ __forceinline__ Meta &meta_of(unsigned char *S, int it) { return *(Meta *)(S + OFF_META + (it & (NM - 1)) * (int)sizeof(Meta)); }

// MN-major operand, 128-byte swizzle: LBO = bytes between 64-element atoms along M/N, SBO = bytes between 8-row groups along K
__device__ __forceinline__ uint64_t desc_mn(uint32_t addr, uint32_t lbo, uint32_t sbo)
{
    return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)((lbo >> 4) & 0x3FFF) << 16) | ((uint64_t)((sbo >> 4) & 0x3FFF) << 32) |
           ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}

// TMA gather of four table rows, 64 bf16 columns starting at `col`, into four consecutive 128-byte rows (swizzled by the map)
__device__ __forceinline__ void gather4(void *dst, const void *tmap, int col, int r0, int r1, int r2, int r3, uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile::gather4.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];"
        ::"r"(tc::smem_u32(dst)), "l"(tmap), "r"(col), "r"(r0), "r"(r1), "r"(r2), "r"(r3), "r"(tc::smem_u32(bar))
        : "memory");
}

// fp32 masters of gfn_node_tc.cu are tile-blocked: [tile of 128 rows][c / 4][row in tile][4 floats]
__device__ __forceinline__ size_t blk_off(int64_t row, int c) { return ((size_t)(row >> 7) * (H / 4) + (c >> 2)) * (128 * 4) + (size_t)(row & 127) * 4 + (c & 3); }

// ---- role P: per-slot geometry (S:G1), K-block row flags, Gaussian basis tile
__device__ __forceinline__ void role_P(const Args &a, unsigned char *S, uint64_t *bar, int n_tiles, int s_begin, int s_end, int p, int lane)
{
    const float inv_rc = 1.0f / a.r_cut;
    const float uc_scale = (float)(K - 1) / a.r_cut * RBF_C;
    const int w = p >> 5;
    for (int it = 0; it < n_tiles; ++it) {
        const int slot = s_begin + it * TP + p;
        const bool valid = slot < s_end;
        int row = -1, cj = -1;
        if (valid) { row = __ldg(a.pair_row + slot); cj = __ldg(a.col + slot); }
        int prev = -3, nxt = -2;
        if (valid && (p & 15) == 0 && slot > s_begin) prev = __ldg(a.pair_row + slot - 1);
        if (valid && (p & 15) == 15 && slot + 1 < s_end) nxt = __ldg(a.pair_row + slot + 1);
        int jrow = valid ? row : 0;
        float wgt = 0.f, dist = 0.f;
        if (cj >= 0) {
            const int sys = row / a.N;
            jrow = sys * a.N + cj;
            float f[3];
#pragma unroll
            for (int ax = 0; ax < 3; ++ax) {      // fp64 difference and minimum image, fp32 from there on
                double dx = a.q[(size_t)jrow * 3 + ax] - a.q[(size_t)row * 3 + ax];
                if (a.periodic) dx = dx - a.box[ax] * rint(dx * a.inv_box[ax]);
                f[ax] = (float)dx;
            }
            const float d2 = fmaf(f[0], f[0], fmaf(f[1], f[1], f[2] * f[2]));
            dist = d2 * rsqrtf(fmaxf(d2, 1e-24f));
            wgt = 0.5f * (cospif(dist * inv_rc) + 1.0f);
        }
        const unsigned sb = __ballot_sync(FULL, valid && (p & 15) == 0 && prev != row);
        const unsigned eb = __ballot_sync(FULL, valid && (p & 15) == 15 && nxt != row);
        // Gaussian basis in registers before the buffers are waited for
        const float uc = dist * uc_scale;         // C d / delta
        uint4 gch[8];
#pragma unroll
        for (int ch = 0; ch < 8; ++ch) {
            float g[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const float t = uc - RBF_C * (float)(ch * 8 + e);
                g[e] = ex2_approx(-t * t);
            }
            gch[ch] = make_uint4(tc::pack_bf16(g[0], g[1]), tc::pack_bf16(g[2], g[3]), tc::pack_bf16(g[4], g[5]), tc::pack_bf16(g[6], g[7]));
        }
        if (w == 1) {                             // poller of role P
            tc::mbar_wait(&bar[META_EMPTY + (it & (NM - 1))], ((it / NM) & 1) ^ 1);
            tc::mbar_wait(&bar[A1_EMPTY], (it & 1) ^ 1);
        }
        tc::named_bar_sync(NB_P, 128);
        Meta &M = meta_of(S, it);
        M.w[p] = wgt; M.jrow[p] = jrow;
        if (lane == 0) M.kflag[w] = (sb & 1u) | ((sb >> 15) & 2u) | (((eb >> 15) & 1u) << 8) | (((eb >> 31) & 1u) << 9);
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(&bar[META_FULL + (it & (NM - 1))]);
        unsigned char *A1 = S + OFF_A1 + p * 128;  // K-major rows of 128 B, 16-byte chunks XOR-swizzled by row & 7
#pragma unroll
        for (int ch = 0; ch < 8; ++ch) *(uint4 *)(A1 + ((ch ^ (p & 7)) << 4)) = gch[ch];
        tc::fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(&bar[A1_FULL]);
    }
}

// ---- role H: c_ij SiLU(2 (D1 + b_e1/2)) -> B planes (bf16), c_ij as a bf16 pair -> first chunk of the third plane.
// Thread p owns TMEM lane p (slot p) and all 128 columns.
__device__ __forceinline__ void role_H(const Args &a, unsigned char *S, uint64_t *bar, uint32_t tmem, int n_tiles, int p, int lane)
{
    const uint32_t td1 = tmem + TM_D1 + ((uint32_t)(p & ~31) << 16);
    for (int it = 0; it < n_tiles; ++it) {
        const int s = it & 1;
        if ((p >> 5) == 2) {                      // poller of role H
            tc::mbar_wait(&bar[B_EMPTY + s], ((it >> 1) & 1) ^ 1);
            tc::mbar_wait(&bar[META_FULL + (it & (NM - 1))], (it / NM) & 1);
            tc::mbar_wait(&bar[D1_FULL], it & 1);
        }
        tc::named_bar_sync(NB_H, 128);
        tc::tc_fence_after_sync();
        const float cw = meta_of(S, it).w[p];
        unsigned char *rowp = S + OFF_B + s * B_STAGE + p * 128;
#pragma unroll
        for (int c2 = 0; c2 < 4; ++c2) {
            uint32_t r0[16], r1[16];
            tc::tmem_ld16_nowait(td1 + c2 * 32, r0);
            tc::tmem_ld16_nowait(td1 + c2 * 32 + 16, r1);
            tc::tmem_ld_wait();
            if (c2 == 3) {                        // D1 is in registers: the next tile's first product may overwrite it
                tc::tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) tc::mbar_arrive(&bar[D1_EMPTY]);
            }
#pragma unroll
            for (int hh = 0; hh < 2; ++hh) {
                const int cc = c2 * 2 + hh;
                uint32_t pk[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int col = cc * 16 + 2 * e;
                    const float h0 = __uint_as_float(hh ? r1[2 * e] : r0[2 * e]) + a.b1h[col];
                    const float h1 = __uint_as_float(hh ? r1[2 * e + 1] : r0[2 * e + 1]) + a.b1h[col + 1];
                    pk[e] = tc::pack_bf16(cw * fmaf(h0, tc::tanh_approx(h0), h0), cw * fmaf(h1, tc::tanh_approx(h1), h1));
                }
                unsigned char *kb = rowp + (cc >> 2) * 16384;
                const int ch0 = (cc & 3) * 2;
                *(uint4 *)(kb + ((ch0 ^ (p & 7)) << 4)) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
                *(uint4 *)(kb + (((ch0 + 1) ^ (p & 7)) << 4)) = make_uint4(pk[4], pk[5], pk[6], pk[7]);
            }
        }
        {   // columns 128, 129 of the N = 144 product: c_ij = hi + lo (bf16 pair); the rest of the plane's first 16 columns stays zero
            const uint32_t hi = tc::pack_bf16(cw, 0.f);
            const uint32_t both = tc::pack_bf16(cw, cw - tc::bf16lo_to_f32(hi));
            *(uint4 *)(rowp + 2 * 16384 + ((0 ^ (p & 7)) << 4)) = make_uint4(both, 0u, 0u, 0u);
        }
        tc::fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) { tc::mbar_arrive(&bar[B_FULL + s]); tc::mbar_arrive(&bar[META_EMPTY + (it & (NM - 1))]); }
    }
}

// ---- role MMA
template <bool FIRST>
__device__ __forceinline__ void role_MMA(const Args &a, unsigned char *S, uint64_t *bar, uint32_t tmem, int n_tiles, int n_slots, int lane)
{
    using C = Cfg<FIRST>;
    constexpr int NR = RING_BYTES / C::STAGE;
    const uint32_t idesc1 = tc::make_idesc_bf16(TP, H);                                      // K-major x K-major
    const uint32_t idescT = tc::make_idesc_bf16(128, 144) | (1u << 15) | (1u << 16);         // MN-major x MN-major
    const uint32_t idesct = tc::make_idesc_bf16(128, 16) | (1u << 15) | (1u << 16);
    const uint32_t sW1 = tc::smem_u32(S + OFF_W1), sA1 = tc::smem_u32(S + OFF_A1), sB = tc::smem_u32(S + OFF_B);
    const uint32_t sR = tc::smem_u32(S + OFF_RING);
    tc::mbar_wait(&bar[W_FULL], 0);
    int g = 0;                  // gather stages consumed
    int acc = 0, nrow = 0;      // accumulator in use, non-empty rows started
    uint32_t accum = 0;
    for (int k = 0; k <= n_tiles; ++k) {
        if (k < n_tiles) {                       // D1 = G (W_e1/2)^T   (4 x UMMA 128x128x16)
            tc::mbar_wait(&bar[D1_EMPTY], (k & 1) ^ 1);
            tc::mbar_wait(&bar[A1_FULL], k & 1);
            tc::tc_fence_after_sync();
            if (lane == 0) {
#pragma unroll
                for (int kk = 0; kk < K / 16; ++kk)
                    tc::mma_bf16_ss(tmem + TM_D1, tc::make_desc_sw128(sA1 + kk * 32), tc::make_desc_sw128(sW1 + kk * 32), idesc1, kk > 0);
                tc::mma_commit(&bar[D1_FULL]);
                tc::mma_commit(&bar[A1_EMPTY]);
            }
            __syncwarp();
        }
        if (k >= 1) {                            // row contraction over the K blocks of tile j
            const int j = k - 1, s = j & 1;
            tc::mbar_wait(&bar[META_FULL + (j & (NM - 1))], (j / NM) & 1);
            tc::mbar_wait(&bar[B_FULL + s], (j >> 1) & 1);
            tc::tc_fence_after_sync();
            const Meta &M = meta_of(S, j);
            unsigned ks = 0, ke = 0;
#pragma unroll
            for (int w = 0; w < 4; ++w) { const unsigned f = M.kflag[w]; ks |= (f & 3u) << (2 * w); ke |= ((f >> 8) & 3u) << (2 * w); }
            const int left = n_slots - j * TP;
            const int nkb = left >= TP ? 8 : (left + 15) / 16;
            const uint32_t sBs = sB + s * B_STAGE;
            for (int kb = 0; kb < nkb; ++kb) {
                const int st = g % NR;
                if ((kb & 1) == 0) {
                    tc::mbar_wait(&bar[RING_FULL + st], (g / NR) & 1);
                    tc::tc_fence_after_sync();
                }
                if ((ks >> kb) & 1u) {           // a row starts: its accumulator must have been drained
                    tc::mbar_wait(&bar[ACC_EMPTY + acc], ((nrow >> 1) & 1) ^ 1);
                    tc::tc_fence_after_sync();
                    accum = 0;
                }
                if (lane == 0) {
                    const uint32_t d = tmem + TM_ACC + acc * ACC_COLS;
                    const uint32_t ax = sR + st * C::STAGE + (kb & 1) * 2048;
                    tc::mma_bf16_ss(d, desc_mn(ax, SB * 128, 1024), desc_mn(sBs + kb * 2048, 16384, 1024), idescT, accum);
                    if (!FIRST)
                        tc::mma_bf16_ss(d + 144, desc_mn(ax + 2 * SB * 128, SB * 128, 1024), desc_mn(sBs + 2 * 16384 + kb * 2048, 16384, 1024), idesct, accum);
                }
                accum = 1;
                if ((ke >> kb) & 1u) {           // the row is complete
                    if (lane == 0) tc::mma_commit(&bar[ACC_FULL + acc]);
                    acc ^= 1; ++nrow;
                }
                if ((kb & 1) == 1 || kb == nkb - 1) {
                    if (lane == 0) tc::mma_commit(&bar[RING_EMPTY + st]);
                    ++g;
                }
                __syncwarp();
            }
            if (lane == 0) { tc::mma_commit(&bar[B_EMPTY + s]); tc::mbar_arrive(&bar[META_EMPTY + (j & (NM - 1))]); }
            __syncwarp();
        }
    }
}

// ---- role G: warp 0 gathers the x planes, warp 1 the y planes, 32 slots per stage
template <bool FIRST>
__device__ __forceinline__ void role_G(const Args &a, unsigned char *S, uint64_t *bar, int n_slots, int gw, int lane)
{
    using C = Cfg<FIRST>;
    constexpr int NR = RING_BYTES / C::STAGE;
    const int n_stages = (n_slots + SB - 1) / SB;
    const int quad = lane & 7, pl = gw * 2 + ((lane >> 3) & 1);
    for (int st = 0; st < n_stages; ++st) {
        const int it = st >> 2, qd = st & 3;
        const Meta &M = meta_of(S, it);
        if (qd == 0) tc::mbar_wait(&bar[META_FULL + (it & (NM - 1))], (it / NM) & 1);
        const int rs = st % NR;
        tc::mbar_wait(&bar[RING_EMPTY + rs], ((st / NR) & 1) ^ 1);
        if (lane == 0) tc::mbar_arrive_expect_tx(&bar[RING_FULL + rs], 2 * SB * 128);
        __syncwarp();
        if (lane < 16) {
            const int4 jr = *(const int4 *)&M.jrow[qd * SB + quad * 4];
            gather4(S + OFF_RING + rs * C::STAGE + pl * (SB * 128) + quad * 512, &a.gmap, pl * 64, jr.x, jr.y, jr.z, jr.w, &bar[RING_FULL + rs]);
        }
        if (qd == 3 || st == n_stages - 1) {
            __syncwarp();
            if (lane == 0) tc::mbar_arrive(&bar[META_EMPTY + (it & (NM - 1))]);
        }
    }
}

// ---- role EPI: thread = channel c.  m_i[c] = agg (W_e2[c][:] . T_i[c][:] + (b[c] + E_i[c]) s_i[c] + t_i[c])
template <bool FIRST>
__device__ __forceinline__ void role_EPI(const Args &a, uint64_t *bar, uint32_t tmem, int r0, int r1, int n_total, int c, int lane)
{
    float Wr[H];
#pragma unroll
    for (int k = 0; k < H; ++k) Wr[k] = __ldg(a.We2T + (size_t)k * H + c);
    const float b2c = __ldg(a.b2 + c);
    const uint32_t base0 = tmem + TM_ACC + ((uint32_t)(c & ~31) << 16);
    int nrow = 0;
    int rp0 = (r0 < r1) ? __ldg(a.row_ptr + r0) : 0;
    for (int row = r0; row < r1; ++row) {
        const int rp1 = __ldg(a.row_ptr + row + 1);
        const int cnt = (n_total > 0) ? rp1 - rp0 : 0;
        rp0 = rp1;
        if (cnt == 0) { a.m_out[(size_t)row * H + c] = 0.f; continue; }
        const int acc = nrow & 1;
        float Ei = 0.f;
        if (!FIRST) Ei = __ldg(a.E + blk_off(row, c));
        if ((c >> 5) == 0) tc::mbar_wait(&bar[ACC_FULL + acc], (nrow >> 1) & 1);
        tc::named_bar_sync(NB_EPI, 128);
        tc::tc_fence_after_sync();
        const uint32_t base = base0 + acc * ACC_COLS;
        float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
#pragma unroll
        for (int k0 = 0; k0 < H; k0 += 32) {
            uint32_t v0[16], v1[16];
            tc::tmem_ld16_nowait(base + k0, v0);
            tc::tmem_ld16_nowait(base + k0 + 16, v1);
            tc::tmem_ld_wait();
#pragma unroll
            for (int e = 0; e < 16; e += 2) {
                s0 = fmaf(Wr[k0 + e], __uint_as_float(v0[e]), s0);
                s1 = fmaf(Wr[k0 + e + 1], __uint_as_float(v0[e + 1]), s1);
                s2 = fmaf(Wr[k0 + 16 + e], __uint_as_float(v1[e]), s2);
                s3 = fmaf(Wr[k0 + 16 + e + 1], __uint_as_float(v1[e + 1]), s3);
            }
        }
        uint32_t vs[16];
        tc::tmem_ld16_nowait(base + 128, vs);
        float tt = 0.f;
        if (!FIRST) {
            uint32_t vt[16];
            tc::tmem_ld16_nowait(base + 144, vt);
            tc::tmem_ld_wait();
            tt = __uint_as_float(vt[0]) + __uint_as_float(vt[1]);
        } else {
            tc::tmem_ld_wait();
        }
        const float ss = __uint_as_float(vs[0]) + __uint_as_float(vs[1]);
        tc::tc_fence_before_sync();
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(&bar[ACC_EMPTY + acc]);
        ++nrow;
        a.m_out[(size_t)row * H + c] = a.agg * (((s0 + s1) + (s2 + s3)) + fmaf(b2c + Ei, ss, tt));
    }
}

template <bool FIRST>
__global__ void __launch_bounds__(THREADS, 1) msg_row_kernel(const __grid_constant__ Args a)
{
    using C = Cfg<FIRST>;
    constexpr int NR = RING_BYTES / C::STAGE;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char *S = smem_raw + ((1024u - (tc::smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t *bar = (uint64_t *)(S + OFF_BAR);
    uint32_t *tmem_slot = (uint32_t *)(S + OFF_TMEM);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int n_total = a.row_ptr[a.rows];
    const int r0 = a.part[blockIdx.x], r1 = a.part[blockIdx.x + 1];
    const int s_begin = (n_total > 0 && r0 < r1) ? a.row_ptr[r0] : 0;
    const int s_end = (n_total > 0 && r0 < r1) ? a.row_ptr[r1] : 0;
    const int n_slots = s_end - s_begin, n_tiles = (n_slots + TP - 1) / TP;

    if (tid == 0) {
        tc::mbar_init(&bar[A1_FULL], 4);  tc::mbar_init(&bar[A1_EMPTY], 1);
        tc::mbar_init(&bar[D1_FULL], 1);  tc::mbar_init(&bar[D1_EMPTY], 4);
        for (int s = 0; s < 2; ++s) {
            tc::mbar_init(&bar[B_FULL + s], 4);   tc::mbar_init(&bar[B_EMPTY + s], 1);
            tc::mbar_init(&bar[ACC_FULL + s], 1); tc::mbar_init(&bar[ACC_EMPTY + s], 4);
        }
        for (int s = 0; s < NM; ++s) { tc::mbar_init(&bar[META_FULL + s], 4); tc::mbar_init(&bar[META_EMPTY + s], 4 + 1 + C::NG); }
        for (int s = 0; s < NR; ++s) { tc::mbar_init(&bar[RING_FULL + s], C::NG); tc::mbar_init(&bar[RING_EMPTY + s], 1); }
        tc::mbar_init(&bar[W_FULL], 1);
        tc::fence_mbar_init();
    }
    if (warp == W_MMA) tc::tmem_alloc(tmem_slot, 512);
    // third B plane (c_ij columns): only the first chunk of each row is ever rewritten; the second chunk must read as zero
    for (int i = tid; i < 2 * 16384 / 16; i += THREADS) {
        const int s = i / 1024, r = i % 1024;
        *(uint4 *)(S + OFF_B + s * B_STAGE + 2 * 16384 + r * 16) = make_uint4(0u, 0u, 0u, 0u);
    }
    tc::fence_proxy_async_smem();
    tc::tc_fence_before_sync();
    __syncthreads();
    tc::tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot;
    if (tid == W_G * 32) {
        tc::mbar_arrive_expect_tx(&bar[W_FULL], 16384);
        tc::bulk_g2s(S + OFF_W1, a.W1img, 16384, &bar[W_FULL]);
    }
    // register re-balancing between the four warpgroups (128 at launch): the epilogue keeps a row of W_e2 in registers
    if (warp < 4) asm volatile("setmaxnreg.dec.sync.aligned.u32 88;");
    else if (warp < 8) asm volatile("setmaxnreg.dec.sync.aligned.u32 88;");
    else if (warp < 12) asm volatile("setmaxnreg.inc.sync.aligned.u32 216;");
    else asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");

    if (warp < W_H) role_P(a, S, bar, n_tiles, s_begin, s_end, tid, lane);
    else if (warp < W_EPI) role_H(a, S, bar, tmem, n_tiles, tid - W_H * 32, lane);
    else if (warp < W_MMA) role_EPI<FIRST>(a, bar, tmem, r0, r1, n_total, tid - W_EPI * 32, lane);
    else if (warp == W_MMA) role_MMA<FIRST>(a, S, bar, tmem, n_tiles, n_slots, lane);
    else if (warp < W_G + C::NG) role_G<FIRST>(a, S, bar, n_slots, warp - W_G, lane);

    tc::tc_fence_before_sync();
    __syncthreads();
    if (warp == W_MMA) tc::tmem_dealloc(tmem, 512);
}

int launch_msg_row(pimd_ctx *c, bool first)
{
    Args a;
    a.gmap = c->tmap_xy;
    a.N = c->N; a.periodic = c->periodic;
    for (int k = 0; k < 3; ++k) { a.box[k] = c->box[k]; a.inv_box[k] = c->periodic ? 1.0 / c->box[k] : 0.0; }
    a.r_cut = c->net.r_cut; a.agg = c->net.agg_norm;
    a.row_ptr = c->nl.row_ptr; a.col = c->nl.col; a.pair_row = c->nl.pair_row; a.part = c->nl.part; a.rows = c->rows; a.q = c->q;
    a.W1img = c->wimg_e1;
    for (int k = 0; k < H; ++k) a.b1h[k] = c->h_be1_half[k];
    a.We2T = c->net.We2T; a.b2 = c->net.be2; a.E = c->Efeat; a.m_out = c->mfeat;
    const size_t smem = SMEM_BYTES + 1024;
    if (!(c->attr_done & ATTR_MSGROW)) {
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(msg_row_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(msg_row_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        c->attr_done |= ATTR_MSGROW;
    }
    if (first) msg_row_kernel<true><<<c->nl.n_part, THREADS, smem, c->stream>>>(a);
    else msg_row_kernel<false><<<c->nl.n_part, THREADS, smem, c->stream>>>(a);
    c->launches++;
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}

}  // namespace gfn_row
