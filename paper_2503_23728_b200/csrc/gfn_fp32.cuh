// gfn_fp32.cuh -- building blocks of the fp32 (FFMA) GFN kernels: 128-row register-tiled GEMM on
// shared-memory operands, swizzled k-major A buffers, activation.
#pragma once
#include "common.cuh"

namespace gfn {

constexpr int TP = 128;   // pairs (or rows) per tile
constexpr int NT = 256;   // threads per CTA
constexpr int TX = 16;    // channel groups per tile

// k-major A buffer [k][TP]; column index XOR-swizzled in units of 4 floats by the k row, so that
// transposing float4 stores from the 16 channel groups hit distinct banks.
__device__ __forceinline__ int swz(int k) { return ((k >> 2) & 7) << 2; }

__device__ __forceinline__ float silu_f(float x) { return __fdividef(x, 1.0f + __expf(-x)); }

template <int H>
struct Tile {
    static constexpr int CPT = H / TX;        // channels per thread (8 for H=128, 4 for H=64)
    static constexpr int NCG = CPT / 4;       // float4 channel groups per thread
    // channel of (group g, element e) for this thread
    __device__ static __forceinline__ int chan(int tx, int g, int e) { return g * (H / 2) + tx * 4 + e; }
    // local pair (row) of (group g, element e)
    __device__ static __forceinline__ int pair(int ty, int g, int e) { return g * (TP / 2) + ty * 4 + e; }
};

// local row of element p of a thread's RP rows (RP = 8: two groups of four, 64 rows apart; 4: one group of four; 2: two rows)
template <int RP>
__device__ __forceinline__ int tile_row(int ty, int p) { return RP == 2 ? ty * 2 + p : (p >> 2) * (TP / 2) + ty * 4 + (p & 3); }

// acc[p][c] += sum_k A[k][p] * W[k][c];  A swizzled [KD][TP], W [KD][H]
// RP = rows per thread: 8 (the whole 128-row tile), 4 or 2 (only rows 0..63 / 0..31 of the buffers are in use: partial tiles for
// configurations with fewer tiles than SMs)
template <int KD, int H, int RP = 8>
__device__ __forceinline__ void tile_gemm(const float *__restrict__ sA, const float *__restrict__ sW,
                                          float (&acc)[RP][Tile<H>::CPT], int tx, int ty)
{
    constexpr int CPT = Tile<H>::CPT;
#pragma unroll 4
    for (int k = 0; k < KD; ++k) {
        const int sw = swz(k);
        float a[RP], b[CPT];
        if constexpr (RP == 2) {
            *(float2 *)&a[0] = *(const float2 *)&sA[k * TP + ((ty * 2) ^ sw)];
        } else {
            *(float4 *)&a[0] = *(const float4 *)&sA[k * TP + ((ty * 4) ^ sw)];
            if constexpr (RP == 8) *(float4 *)&a[RP - 4] = *(const float4 *)&sA[k * TP + ((TP / 2 + ty * 4) ^ sw)];
        }
        *(float4 *)&b[0] = *(const float4 *)&sW[k * H + tx * 4];
        if (CPT == 8) *(float4 *)&b[CPT - 4] = *(const float4 *)&sW[k * H + H / 2 + tx * 4];
#pragma unroll
        for (int p = 0; p < RP; ++p)
#pragma unroll
            for (int c = 0; c < CPT; ++c) acc[p][c] = fmaf(a[p], b[c], acc[p][c]);
    }
}

template <int H, int RP = 8>
__device__ __forceinline__ void zero_acc(float (&acc)[RP][Tile<H>::CPT])
{
#pragma unroll
    for (int p = 0; p < RP; ++p)
#pragma unroll
        for (int c = 0; c < Tile<H>::CPT; ++c) acc[p][c] = 0.f;
}

// writes v[p][c] (this thread's 8 x CPT sub-tile) into a swizzled k-major buffer as A[c][p]
template <int H, int RP = 8>
__device__ __forceinline__ void store_as_A(float *sA, const float (&v)[RP][Tile<H>::CPT], int tx, int ty)
{
    constexpr int CPT = Tile<H>::CPT;
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
        const int ch = Tile<H>::chan(tx, c >> 2, c & 3);
        const int sw = swz(ch);
        if constexpr (RP == 2) {
            *(float2 *)&sA[ch * TP + ((ty * 2) ^ sw)] = make_float2(v[0][c], v[1][c]);
        } else {
            *(float4 *)&sA[ch * TP + ((ty * 4) ^ sw)] = make_float4(v[0][c], v[1][c], v[2][c], v[3][c]);
            if constexpr (RP == 8) *(float4 *)&sA[ch * TP + ((TP / 2 + ty * 4) ^ sw)] = make_float4(v[RP - 4][c], v[RP - 3][c], v[RP - 2][c], v[RP - 1][c]);
        }
    }
}

// cooperative copy of a [rows][H] fp32 matrix from global into shared memory
template <int H>
__device__ __forceinline__ void load_matrix(float *sW, const float *__restrict__ g, int rows)
{
    const float4 *g4 = (const float4 *)g;
    float4 *s4 = (float4 *)sW;
    for (int i = threadIdx.x; i < rows * H / 4; i += NT) s4[i] = __ldg(g4 + i);
}

}  // namespace gfn
