// gfn_node_tc.cu -- atom-wise dense layers of the GFN force net on the 5th-gen tensor cores
// (rows a4, a6 of SURVEY 8(a); P:L74 phi_v and the node->edge MLP of P:L76), bf16 operands with fp32
// accumulation in TMEM.  Used when gemm_dtype == 1 and H == 128 (BASELINE configs[3..4]).
//
// Per 128-row tile and layer:
//   h   = SiLU(W_vn n + W_vm m + b_v1)      one K = 256 accumulation chain, m assembled from the carry slots
//   n  += W_v2 h + b_v2                     fp32 residual stream in HBM
//   E  += W_a n + b_a                       running sum of the edge updates (S:G5), fp32 master in HBM
//   x   = W_s^{l+1} n                       or, after the last layer,  G = W_f1 E
// Precision (tests/test_bf16_emulation.py): a plain bf16 operand carries a rounding error of up to
// 2^-8 relative, and the emulation shows that the atom-wise products alone then move the forces by about 1 % rms and 2 % per atom
// of rms|F| (mostly through the rounded WEIGHTS, then the E path W_a, W_f1) -- all of north_star's 2e-2.  So every operand
// of these products is carried as a bf16 PAIR v = hi + lo (hi = bf16(v), lo = bf16(v - hi)) and a product is three bf16
// tensor-core products A_hi W_hi + A_lo W_hi + A_hi W_lo accumulated in fp32 (error <= 2^-16 per operand); only x = W_s n is
// a single product, because x is gathered as bf16 by the message pass anyway.  The tensor pipe has the time (the kernel is
// bound by its HBM reads and writes); shared memory does not hold ten 32 KB weight images, so the weight images stream
// from L2 through a ring of 16 KB slots (TMA bulk copies, one producer warp), 18 (20 in the last layer) slots per tile.
// The pair kernels gather x_j and y_j = E_j x_j per directed pair in the message passes: that copy is one 32-bit word per
// channel (XE[row][c]: x as bf16 in the low half; the whole word read as fp32 is y to half a bf16 ulp, tc::pack_x_y), so one
// load serves both and the L2 gather traffic halves.  G stays fp32:
// G_i + G_j enters the force readout directly, with no averaging over neighbours behind it.
// SiLU(x) = h tanh(h) + h with h = x/2: the 1/2 is folded (exactly) into the W_vn, W_vm images and b_v1.
#include "common.cuh"
#include "tc_ptx.cuh"

namespace node_tc {

constexpr int TR = 128;            // rows per tile
constexpr int H = 128;
constexpr int NCW = 16;            // compute warps (load, epilogues); warp 16 is the weight producer
constexpr int NTC = NCW * 32;
constexpr int NTH = NTC + 32;
constexpr int OPB = TR * H * 2;    // bytes of one bf16 operand tile
constexpr int SLOT = 16384;        // one K block (64 k) of a weight image: [128 n][64 k] bf16, 128-byte swizzle
constexpr int NS = 5;              // ring slots
// half-images per layer in the order the tile consumes them: (W_vn/2, W_vm/2, W_v2, W_a) x (hi, lo) x 2 K blocks, then
// W_next hi (x of the next layer: one product) or, in the last layer, W_f1 hi and lo
constexpr int SEQ_MID = 18, SEQ_LAST = 20, IMG_PER_LAYER = 20;

struct Args {
    int64_t rows;
    int N, last, gran_m, n_tiles;
    const int *row_ptr;
    const uint16_t *Wimg;          // this layer's IMG_PER_LAYER half-images, SLOT bytes each
    const float *bv1, *bv2, *ba;
    float *n, *E;
    const float *m, *carry_m;
    uint32_t *XE;
    float *G;
};

constexpr int OFF_RING = 0, OFF_A0H = NS * SLOT, OFF_A0L = OFF_A0H + OPB, OFF_A1H = OFF_A0L + OPB, OFF_A1L = OFF_A1H + OPB,
              OFF_B = OFF_A1L + OPB, OFF_BAR = OFF_B + 3 * H * 4, SMEM_BYTES = OFF_BAR + (2 * NS + 1) * 8 + 16;
constexpr int NB_COMPUTE = 1;      // named barrier of the 16 compute warps (0 would include the producer warp)

// byte offset of element (row r, k) in a K-major [128][128] bf16 operand: two k-blocks of [128][64] (128-byte rows),
// 16-byte chunks XOR-swizzled by r & 7
__device__ __forceinline__ int op_off(int r, int k)
{
    return (k >> 6) * (TR * 128) + r * 128 + ((((k & 63) >> 3) ^ (r & 7)) << 4) + (k & 7) * 2;
}

// fp32 masters n and E are private to these kernels and kept tile-blocked: [tile][c / 4][row in tile][4 floats], so that the
// epilogue, where a thread owns a row (TMEM lane), reads and writes 512 contiguous bytes per warp instruction.
__device__ __forceinline__ size_t blk_off(int64_t row0, int r, int c) { return ((size_t)(row0 >> 7) * (H / 4) + (c >> 2)) * (TR * 4) + (size_t)r * 4 + (c & 3); }

// v = hi + lo with hi = bf16(v), lo = bf16(v - hi): packed pairs (a, b) -> (hi word, lo word)
__device__ __forceinline__ void split2(float a, float b, uint32_t &hi, uint32_t &lo)
{
    hi = tc::pack_bf16(a, b);
    lo = tc::pack_bf16(a - tc::bf16lo_to_f32(hi), b - tc::bf16hi_to_f32(hi));
}

// 16 fp32 values of row r, columns [c0, c0 + 16) -> bf16 hi / lo -> two swizzled 16-byte chunks of each operand tile
__device__ __forceinline__ void store_operand16(unsigned char *Ah, unsigned char *Al, int r, int c0, const float (&v)[16])
{
    uint32_t ph[8], pl[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) split2(v[2 * e], v[2 * e + 1], ph[e], pl[e]);
    const int base = (c0 >> 6) * (TR * 128) + r * 128;
    const int ch = (c0 & 63) >> 3;
    const int o0 = base + ((ch ^ (r & 7)) << 4), o1 = base + (((ch + 1) ^ (r & 7)) << 4);
    *(uint4 *)(Ah + o0) = make_uint4(ph[0], ph[1], ph[2], ph[3]);
    *(uint4 *)(Ah + o1) = make_uint4(ph[4], ph[5], ph[6], ph[7]);
    *(uint4 *)(Al + o0) = make_uint4(pl[0], pl[1], pl[2], pl[3]);
    *(uint4 *)(Al + o1) = make_uint4(pl[4], pl[5], pl[6], pl[7]);
}

__device__ __forceinline__ void store_operand4(unsigned char *Ah, unsigned char *Al, int r, int k, float4 v)
{
    uint32_t h0, l0, h1, l1;
    split2(v.x, v.y, h0, l0);
    split2(v.z, v.w, h1, l1);
    const int o = op_off(r, k);
    *(uint2 *)(Ah + o) = make_uint2(h0, h1);
    *(uint2 *)(Al + o) = make_uint2(l0, l1);
}

// the MMA thread's walk through the weight ring: slot g % NS holds half-image number g of this CTA's sequence
struct Ring {
    uint64_t *full, *empty;
    uint32_t sRing;
    uint32_t g;
    // D (+)= A[kb] . W_slot^T for one K block (4 x UMMA 128x128x16); A given as hi (and lo when `both`) operand tiles
    __device__ __forceinline__ void consume(uint32_t tmem_d, uint32_t sAh, uint32_t sAl, int kb, bool both, uint32_t idesc, bool &acc)
    {
        const uint32_t slot = g % NS;
        tc::mbar_wait(&full[slot], (g / NS) & 1);
        tc::tc_fence_after_sync();
        const uint32_t sW = sRing + slot * SLOT, aoff = kb * (TR * 128);
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
            tc::mma_bf16_ss(tmem_d, tc::make_desc_sw128(sAh + aoff + kk * 32), tc::make_desc_sw128(sW + kk * 32), idesc, acc ? 1u : 0u);
            acc = true;
        }
        if (both)
#pragma unroll
            for (int kk = 0; kk < 4; ++kk)
                tc::mma_bf16_ss(tmem_d, tc::make_desc_sw128(sAl + aoff + kk * 32), tc::make_desc_sw128(sW + kk * 32), idesc, 1u);
        tc::mma_commit(&empty[slot]);      // slot free once these products have read it
        ++g;
    }
    // A W^T with A = Ah + Al and W = W_hi + W_lo (four half-images: hi kb0, hi kb1, lo kb0, lo kb1): A_hi W_hi + A_lo W_hi + A_hi W_lo
    __device__ __forceinline__ void product3(uint32_t tmem_d, uint32_t sAh, uint32_t sAl, uint32_t idesc, bool &acc)
    {
        consume(tmem_d, sAh, sAl, 0, true, idesc, acc);
        consume(tmem_d, sAh, sAl, 1, true, idesc, acc);
        consume(tmem_d, sAh, sAl, 0, false, idesc, acc);
        consume(tmem_d, sAh, sAl, 1, false, idesc, acc);
    }
};

__global__ void __launch_bounds__(NTH, 1) node_tc_kernel(const __grid_constant__ Args a)
{ pdl_enter();
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char *S = smem_raw + ((1024u - (tc::smem_u32(smem_raw) & 1023u)) & 1023u);
    unsigned char *A0h = S + OFF_A0H, *A0l = S + OFF_A0L, *A1h = S + OFF_A1H, *A1l = S + OFF_A1L;
    float *sb = (float *)(S + OFF_B);
    uint64_t *bar_full = (uint64_t *)(S + OFF_BAR), *bar_empty = bar_full + NS, *mbar_mma = bar_empty + NS;
    uint32_t *tmem_slot = (uint32_t *)(mbar_mma + 1);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int n_pairs = a.row_ptr[a.rows];
    const int n_seq = a.last ? SEQ_LAST : SEQ_MID;

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { tc::mbar_init(&bar_full[s], 1); tc::mbar_init(&bar_empty[s], 1); }
        tc::mbar_init(mbar_mma, 1);
        tc::fence_mbar_init();
    }
    if (warp == 1) tc::tmem_alloc(tmem_slot, 256);
    for (int i = tid; i < H; i += NTH) { sb[i] = 0.5f * a.bv1[i]; sb[H + i] = a.bv2[i]; sb[2 * H + i] = a.ba[i]; }
    tc::tc_fence_before_sync();
    __syncthreads();
    tc::tc_fence_after_sync();

    if (warp == NCW) {
        // ---- weight producer: the layer's half-images, in consumption order, once per tile of this CTA
        if (lane == 0) {
            uint32_t g = 0;
            for (int tile = blockIdx.x; tile < a.n_tiles; tile += gridDim.x)
                for (int s = 0; s < n_seq; ++s, ++g) {
                    const uint32_t slot = g % NS;
                    tc::mbar_wait(&bar_empty[slot], ((g / NS) & 1) ^ 1);
                    tc::mbar_arrive_expect_tx(&bar_full[slot], SLOT);
                    // mid layers skip W_next lo: image 16, 17 are W_next hi in both cases
                    tc::bulk_g2s(S + OFF_RING + slot * SLOT, a.Wimg + (size_t)s * (SLOT / 2), SLOT, &bar_full[slot]);
                }
        }
        return;                                    // TMEM is freed by warp 1 after the compute warps' last barrier
    }

    const uint32_t tmem_d0 = *tmem_slot, tmem_d1 = tmem_d0 + 128;
    const int q = warp & 3, g = warp >> 2;                 // TMEM lane quadrant; 32-column group
    const int r = q * 32 + lane;                           // row of the tile = TMEM lane
    const uint32_t lane_field = (uint32_t)(q * 32) << 16;
    const uint32_t idesc = tc::make_idesc_bf16(TR, H);
    const uint32_t sA0h = tc::smem_u32(A0h), sA0l = tc::smem_u32(A0l), sA1h = tc::smem_u32(A1h), sA1l = tc::smem_u32(A1l);
    Ring ring{bar_full, bar_empty, tc::smem_u32(S + OFF_RING), 0u};
    uint32_t par = 0;

    for (int tile = blockIdx.x; tile < a.n_tiles; tile += gridDim.x) {
        const int64_t row0 = (int64_t)tile * TR;
        // ---- operands n, m (fp32 in HBM) -> bf16 hi/lo swizzled tiles; m: one warp per row, coalesced 512-byte reads.
        // m_i is assembled in fixed order from the direct row or the carry slots (tail slot of the first granule, head
        // slots of the rest).  All loads of four rows are issued before the first use: the phase is latency-bound.
        {
            // n: the masters are tile-blocked ([c / 4][row][4 floats]), so with thread = row a warp reads 512 contiguous bytes
            // per instruction; eight loads in flight per thread (columns cgrp * 32 .. + 31), issued before everything else
            {
                const int nr = tid & 127, cgrp = tid >> 7;
                const bool nok = row0 + nr < a.rows;
                float4 nv8[8];
#pragma unroll
                for (int i = 0; i < 8; ++i)
                    nv8[i] = nok ? *(const float4 *)(a.n + blk_off(row0, nr, cgrp * 32 + i * 4)) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                for (int i = 0; i < 8; ++i) store_operand4(A0h, A0l, nr, cgrp * 32 + i * 4, nv8[i]);
            }
            const int k = lane * 4, wrow = tid >> 5;
            int rs[8], re[8];
#pragma unroll
            for (int it = 0; it < 8; ++it) {
                const int64_t row = row0 + wrow + it * 16;
                const bool ok = row < a.rows && n_pairs > 0;
                rs[it] = ok ? __ldg(a.row_ptr + row) : 0;
                re[it] = ok ? __ldg(a.row_ptr + row + 1) : 0;
            }
#pragma unroll
            for (int it0 = 0; it0 < 8; it0 += 4) {
                float4 pc[4][4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int it = it0 + j;
                    const int64_t row = row0 + wrow + it * 16;
                    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
                    pc[j][0] = pc[j][1] = pc[j][2] = pc[j][3] = z;
                    if (re[it] > rs[it]) {       // warp-uniform
                        const int g0 = rs[it] / a.gran_m, g1 = (re[it] - 1) / a.gran_m;
                        if (g0 == g1) pc[j][0] = __ldg((const float4 *)(a.m + (size_t)row * H + k));
                        else pc[j][0] = __ldg((const float4 *)(a.carry_m + ((size_t)g0 * 2 + 1) * H + k));
#pragma unroll
                        for (int t = 1; t < 4; ++t)
                            if (g0 + t <= g1) pc[j][t] = __ldg((const float4 *)(a.carry_m + ((size_t)(g0 + t) * 2) * H + k));
                    }
                }
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int it = it0 + j, rr = wrow + it * 16;
                    float4 mv = pc[j][0];
#pragma unroll
                    for (int t = 1; t < 4; ++t) { mv.x += pc[j][t].x; mv.y += pc[j][t].y; mv.z += pc[j][t].z; mv.w += pc[j][t].w; }
                    if (re[it] > rs[it]) {       // rows with more than four granules (very long rows): the rest, in order
                        const int g0 = rs[it] / a.gran_m, g1 = (re[it] - 1) / a.gran_m;
                        for (int gg = g0 + 4; gg <= g1; ++gg) {
                            const float4 t4 = __ldg((const float4 *)(a.carry_m + ((size_t)gg * 2) * H + k));
                            mv.x += t4.x; mv.y += t4.y; mv.z += t4.z; mv.w += t4.w;
                        }
                    }
                    store_operand4(A1h, A1l, rr, k, mv);
                }
            }
        }
        tc::fence_proxy_async_smem();
        tc::named_bar_sync(NB_COMPUTE, NTC);
        // ---- D0 = n (W_vn/2)^T + m (W_vm/2)^T
        if (tid == 0) {
            tc::tc_fence_after_sync();
            bool acc = false;
            ring.product3(tmem_d0, sA0h, sA0l, idesc, acc);
            ring.product3(tmem_d0, sA1h, sA1l, idesc, acc);
            tc::mma_commit(mbar_mma);
        }
        tc::mbar_wait(mbar_mma, par);
        par ^= 1;
        tc::tc_fence_after_sync();
        // ---- h = SiLU(2 (D0 + b_v1/2)) -> A1
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int c0 = g * 32 + j * 16;
            float v[16];
            tc::tmem_ld16(tmem_d0 + lane_field + c0, v);
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                const float hh = v[e] + sb[c0 + e];
                v[e] = fmaf(hh, tc::tanh_approx(hh), hh);
            }
            store_operand16(A1h, A1l, r, c0, v);
        }
        tc::tc_fence_before_sync();
        tc::fence_proxy_async_smem();
        tc::named_bar_sync(NB_COMPUTE, NTC);
        // ---- D0 = h W_v2^T
        if (tid == 0) {
            tc::tc_fence_after_sync();
            bool acc = false;
            ring.product3(tmem_d0, sA1h, sA1l, idesc, acc);
            tc::mma_commit(mbar_mma);
        }
        tc::mbar_wait(mbar_mma, par);
        par ^= 1;
        tc::tc_fence_after_sync();
        // ---- n <- n + D0 + b_v2  (fp32 master in HBM; bf16 hi/lo copy -> A0)
        const int64_t row = row0 + r;
        const bool valid = row < a.rows;
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int c0 = g * 32 + j * 16;
            float v[16], nn[16];
            tc::tmem_ld16(tmem_d0 + lane_field + c0, v);
#pragma unroll
            for (int e4 = 0; e4 < 4; ++e4) {
                float4 t = valid ? *(const float4 *)(a.n + blk_off(row0, r, c0 + e4 * 4)) : make_float4(0.f, 0.f, 0.f, 0.f);
                nn[e4 * 4 + 0] = t.x; nn[e4 * 4 + 1] = t.y; nn[e4 * 4 + 2] = t.z; nn[e4 * 4 + 3] = t.w;
            }
#pragma unroll
            for (int e = 0; e < 16; ++e) nn[e] = nn[e] + (v[e] + sb[H + c0 + e]);
            if (valid)
#pragma unroll
                for (int e4 = 0; e4 < 4; ++e4)
                    *(float4 *)(a.n + blk_off(row0, r, c0 + e4 * 4)) =
                        make_float4(nn[e4 * 4], nn[e4 * 4 + 1], nn[e4 * 4 + 2], nn[e4 * 4 + 3]);
            store_operand16(A0h, A0l, r, c0, nn);
        }
        tc::tc_fence_before_sync();
        tc::fence_proxy_async_smem();
        tc::named_bar_sync(NB_COMPUTE, NTC);
        // ---- D0 = n W_a^T ;  D1 = n W_next^T (x of the next layer: one bf16 product, x is gathered as bf16)
        if (tid == 0) {
            tc::tc_fence_after_sync();
            bool acc = false;
            ring.product3(tmem_d0, sA0h, sA0l, idesc, acc);
            if (!a.last) {
                bool acc1 = false;
                ring.consume(tmem_d1, sA0h, sA0l, 0, false, idesc, acc1);
                ring.consume(tmem_d1, sA0h, sA0l, 1, false, idesc, acc1);
            }
            tc::mma_commit(mbar_mma);
        }
        tc::mbar_wait(mbar_mma, par);
        par ^= 1;
        tc::tc_fence_after_sync();
        // ---- E <- E + D0 + b_a ; XE = x (bf16, low half) with y = E x in the whole word (tc::pack_x_y), or E -> A1 for G = W_f1 E
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int c0 = g * 32 + j * 16;
            float v[16], ee[16];
            tc::tmem_ld16(tmem_d0 + lane_field + c0, v);
#pragma unroll
            for (int e4 = 0; e4 < 4; ++e4) {
                float4 t = valid ? *(const float4 *)(a.E + blk_off(row0, r, c0 + e4 * 4)) : make_float4(0.f, 0.f, 0.f, 0.f);
                ee[e4 * 4 + 0] = t.x; ee[e4 * 4 + 1] = t.y; ee[e4 * 4 + 2] = t.z; ee[e4 * 4 + 3] = t.w;
            }
#pragma unroll
            for (int e = 0; e < 16; ++e) ee[e] = ee[e] + (v[e] + sb[2 * H + c0 + e]);
            if (valid)
#pragma unroll
                for (int e4 = 0; e4 < 4; ++e4)
                    *(float4 *)(a.E + blk_off(row0, r, c0 + e4 * 4)) =
                        make_float4(ee[e4 * 4], ee[e4 * 4 + 1], ee[e4 * 4 + 2], ee[e4 * 4 + 3]);
            if (!a.last) {
                tc::tmem_ld16(tmem_d1 + lane_field + c0, v);
                // A thread owns a row, so a direct store is 16 bytes per lane at a 512-byte stride (32 sectors per
                // instruction).  The warp's 32 x 128-byte block goes through shared memory instead (the operand tiles
                // are free now; 16-byte chunks XOR-swizzled by row & 7) and leaves as whole 128-byte lines below.
                unsigned char *xs = A0h + warp * 4096 + lane * 128;
#pragma unroll
                for (int e4 = 0; e4 < 4; ++e4)
                    *(uint4 *)(xs + (((j * 4 + e4) ^ (lane & 7)) << 4)) =
                        make_uint4(tc::pack_x_y(v[e4 * 4], ee[e4 * 4]), tc::pack_x_y(v[e4 * 4 + 1], ee[e4 * 4 + 1]),
                                   tc::pack_x_y(v[e4 * 4 + 2], ee[e4 * 4 + 2]), tc::pack_x_y(v[e4 * 4 + 3], ee[e4 * 4 + 3]));
            } else {
                store_operand16(A1h, A1l, r, c0, ee);
            }
        }
        if (!a.last) {             // the warp's XE block: 4 rows x 128 bytes per store instruction
            __syncwarp();
#pragma unroll
            for (int it = 0; it < 8; ++it) {
                const int rr = it * 4 + (lane >> 3), ch = lane & 7;
                const uint4 w4 = *(const uint4 *)(A0h + warp * 4096 + rr * 128 + ((ch ^ (rr & 7)) << 4));
                const int64_t orow = row0 + q * 32 + rr;
                if (orow < a.rows) *(uint4 *)(a.XE + (size_t)orow * H + g * 32 + ch * 4) = w4;
            }
        }
        if (a.last) {
            tc::tc_fence_before_sync();
            tc::fence_proxy_async_smem();
            tc::named_bar_sync(NB_COMPUTE, NTC);
            if (tid == 0) {
                tc::tc_fence_after_sync();
                bool acc = false;
                ring.product3(tmem_d1, sA1h, sA1l, idesc, acc);
                tc::mma_commit(mbar_mma);
            }
            tc::mbar_wait(mbar_mma, par);
            par ^= 1;
            tc::tc_fence_after_sync();
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int c0 = g * 32 + j * 16;
                float v[16];
                tc::tmem_ld16(tmem_d1 + lane_field + c0, v);
                // through shared memory like XE (the A0 tiles are free: every product that read them has completed), whole 128-byte lines to HBM
                unsigned char *xs = A0h + warp * 4096 + lane * 128;
#pragma unroll
                for (int e4 = 0; e4 < 4; ++e4)
                    *(float4 *)(xs + (((j * 4 + e4) ^ (lane & 7)) << 4)) = make_float4(v[e4 * 4], v[e4 * 4 + 1], v[e4 * 4 + 2], v[e4 * 4 + 3]);
            }
            __syncwarp();
#pragma unroll
            for (int it = 0; it < 8; ++it) {
                const int rr = it * 4 + (lane >> 3), ch = lane & 7;
                const float4 w4 = *(const float4 *)(A0h + warp * 4096 + rr * 128 + ((ch ^ (rr & 7)) << 4));
                const int64_t orow = row0 + q * 32 + rr;
                if (orow < a.rows) *(float4 *)(a.G + (size_t)orow * H + g * 32 + ch * 4) = w4;
            }
        }
        tc::tc_fence_before_sync();
        tc::named_bar_sync(NB_COMPUTE, NTC);   // TMEM and operand tiles free for the next tile
    }
    if (warp == 1) tc::tmem_dealloc(tmem_d0, 256);
}

// layer-0 inputs: n = Emb[species], E = 0, x = W_s^0 n (one vector per species, formed on the host) -> XE
__global__ void node_init_tc_kernel(int64_t rows, int N, const int *__restrict__ species, const float *__restrict__ Emb,
                                    const float *__restrict__ xs0, float *__restrict__ n, float *__restrict__ E,
                                    uint32_t *__restrict__ XE)
{ pdl_enter();
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;      // over the rows rounded up to whole tiles
    {   // tile-blocked masters: consecutive threads = consecutive rows of one 4-column group (16 contiguous bytes each)
        const int64_t tile = idx >> 12;
        const int c0 = (int)((idx >> 7) & 31) * 4;
        const int64_t row = tile * 128 + (idx & 127);
        if (row < rows) {
            const float4 nv = __ldg((const float4 *)(Emb + (size_t)species[row % N] * H + c0));
            const size_t o = blk_off(tile * 128, (int)(idx & 127), c0);
            *(float4 *)(n + o) = nv;
            *(float4 *)(E + o) = make_float4(0.f, 0.f, 0.f, 0.f);
        }
    }
    // row-major XE: consecutive threads = consecutive columns of one row
    if (idx >= rows * (H / 4)) return;
    const int64_t row = idx >> 5;
    const int c0 = (int)(idx & 31) * 4;
    const float4 xv = __ldg((const float4 *)(xs0 + (size_t)species[row % N] * H + c0));
    *(uint4 *)(XE + (size_t)row * H + c0) =
        make_uint4(tc::pack_bf16(xv.x, 0.f), tc::pack_bf16(xv.y, 0.f), tc::pack_bf16(xv.z, 0.f), tc::pack_bf16(xv.w, 0.f));
}

int launch_node_tc(pimd_ctx *c, int mode, int layer)
{
    const GfnDev &n = c->net;
    if (mode == 0) {
        const int64_t work = (c->rows + 127) / 128 * 128 * (H / 4);
        pimd_launch(node_init_tc_kernel, (unsigned)((work + 255) / 256), 256, 0, c->stream, c->rows, c->N, c->species, n.Emb, c->xs0,
                                                                                 c->nfeat, c->Efeat, c->XE);
        c->launches++;
        PIMD_CUDA_CHECK(cudaGetLastError());
        return 0;
    }
    const GfnLayerW &w = n.layer[layer];
    Args a;
    a.rows = c->rows; a.N = c->N; a.last = (layer == n.L - 1); a.gran_m = c->gran_m;
    a.n_tiles = (int)((c->rows + TR - 1) / TR);
    a.row_ptr = c->nl.row_ptr;
    a.Wimg = c->wimg_node + (size_t)layer * IMG_PER_LAYER * (SLOT / 2);
    a.bv1 = w.bv1; a.bv2 = w.bv2; a.ba = w.ba;
    a.n = c->nfeat; a.E = c->Efeat; a.m = c->mfeat; a.carry_m = c->carry_m;
    a.XE = c->XE; a.G = c->Gfeat;
    const size_t smem = SMEM_BYTES + 1024;
    if (!(c->attr_done & ATTR_NODETC)) {
        PIMD_CUDA_CHECK(cudaFuncSetAttribute(node_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        c->attr_done |= ATTR_NODETC;
    }
    const int grid = a.n_tiles < c->num_sms ? a.n_tiles : c->num_sms;
    pimd_launch(node_tc_kernel, grid, NTH, smem, c->stream, a);
    c->launches++;
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}

}  // namespace node_tc
