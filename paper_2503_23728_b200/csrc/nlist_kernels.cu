// nlist_kernels.cu -- per-bead-system periodic cell list -> CSR pair list (rows a1-a3 of SURVEY 8(a)), with
// neighbour-list reuse (the paper fixes only the cutoff): the cell-list pass collects CANDIDATES
// within r_cut + skin at reference positions and is repeated only when some atom has moved by skin/2 or more since
// (decided on the device, no host synchronisation: the rebuild kernels are launched every step and return at once when
// the flag is clear); every step the exact list is filtered from the candidates with the same fp64 predicate S:L3, so
// the CSR, and with it the forces, are identical to a rebuild from scratch.  skin = 0 rebuilds every step.
//
// bin (wrapped fraction -> cell) -> counting sort (histogram, per-system exclusive scan, scatter of atom index + fp64
// position into cell order) -> one CTA per cell stages its de-duplicated 3x3x3 stencil in shared memory (fp32 coordinates
// relative to the cell's first atom); a lane is a home atom, the four warps share the candidates; an fp32 estimate of d^2
// settles every candidate outside a 1e-3 band around r_c^2 and the exact fp64 sequence of S:L3 (explicit round-to-nearest
// intrinsics, no FMA contraction) decides inside it, so the list is bit-identical to the oracle's; hits are parked in a
// fixed-stride scratch row -> row_ptr scan -> fill through a per-warp bitmask over the atoms of the system, which emits
// every CSR row in ascending j without a sort.  Integer atomics only order the scratch; the CSR is deterministic.
#include "common.cuh"

namespace {

struct NlArgs {
    int N, nsys, periodic;
    int64_t rows;
    double box[3], inv_box[3];     // inv_box = 1 / box (0 when not periodic)
    double rc2;
    double rl2;                    // (r_cut + skin)^2: candidate radius of the cell-list pass
    float rc2_lo, rc2_hi;          // fp32 pre-filter band around the candidate radius^2 (exact fp64 test inside the band)
    double skin_half2;             // (skin / 2)^2
    const int *need;               // device flag: 1 = the candidate lists must be rebuilt this step
    int *need_w;
    float boxf[3], inv_boxf[3];
    int nc[3], nct, hit_stride;
    const double *q;
    NlistDev d;
    int *err;
};

// displacement since the candidate lists were built: any atom at or beyond skin/2 raises the rebuild flag
__global__ void verlet_check_kernel(NlArgs a)
{ pdl_enter();
    int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= a.rows) return;
    double d2 = 0.0;
    const double x[3] = {a.q[row * 3], a.q[row * 3 + 1], a.q[row * 3 + 2]};
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) { const double d = x[ax] - a.d.q_ref[row * 3 + ax]; d2 += d * d; }
    if (!(d2 < a.skin_half2)) *a.need_w = 1;       // (also NaN positions)
    a.d.q32[row] = make_float4((float)x[0], (float)x[1], (float)x[2], 0.f);   // fp32 copy for the filter's estimate (one 16-byte gather per candidate)
}

__global__ void bin_kernel(NlArgs a)
{ pdl_enter();
    if (!*a.need) return;
    int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= a.rows) return;
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) a.d.q_ref[row * 3 + ax] = a.q[row * 3 + ax];   // reference positions of the new candidate lists
    if (row == 0) a.need_w[1] += 1;                                              // rebuild counter (pimd_nlist_rebuilds)
    int cell = 0;
    if (a.periodic) {
        int c[3];
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) {
            double x = a.q[row * 3 + ax] / a.box[ax];
            double f = x - floor(x);
            int ci = (int)(f * a.nc[ax]);
            if (ci > a.nc[ax] - 1) ci = a.nc[ax] - 1;
            if (ci < 0) ci = 0;   // NaN positions
            c[ax] = ci;
        }
        cell = (c[0] * a.nc[1] + c[1]) * a.nc[2] + c[2];
    }
    a.d.cell_id[row] = cell;
    int sys = (int)(row / a.N);
    atomicAdd(&a.d.cell_count[(size_t)sys * a.nct + cell], 1);
}

// block-wide exclusive scan of one value per thread (blockDim.x multiple of 32, <= 1024)
__device__ __forceinline__ int block_exclusive_scan(int v, int *total)
{
    __shared__ int warp_tot[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) warp_tot[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int w = (lane < nw) ? warp_tot[lane] : 0, winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += t;
        }
        warp_tot[lane] = winc - w;  // exclusive warp offsets
        if (lane == 31) *total = winc;
    }
    __syncthreads();
    int res = warp_tot[wid] + inc - v;
    __syncthreads();
    return res;
}

// one block per bead-system: cell_start (relative) = exclusive scan of cell_count; zero the cursors
__global__ void __launch_bounds__(256) scan_cells_kernel(NlArgs a)
{ pdl_enter();
    if (!*a.need) return;
    __shared__ int tot;
    const int sys = blockIdx.x;
    const int *cnt = a.d.cell_count + (size_t)sys * a.nct;
    int *start = a.d.cell_start + (size_t)sys * (a.nct + 1);
    int *cur = a.d.cell_cursor + (size_t)sys * a.nct;
    int carry = 0;
    for (int base = 0; base < a.nct; base += blockDim.x) {
        int c = base + threadIdx.x;
        int v = (c < a.nct) ? cnt[c] : 0;
        int ex = block_exclusive_scan(v, &tot);
        if (c < a.nct) { start[c] = carry + ex; cur[c] = 0; }
        carry += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) start[a.nct] = carry;
}

__global__ void scatter_kernel(NlArgs a)
{ pdl_enter();
    if (!*a.need) return;
    int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= a.rows) return;
    int sys = (int)(row / a.N), i = (int)(row - (int64_t)sys * a.N);
    int cell = a.d.cell_id[row];
    int slot = atomicAdd(&a.d.cell_cursor[(size_t)sys * a.nct + cell], 1);
    int64_t pos = (int64_t)sys * a.N + a.d.cell_start[(size_t)sys * (a.nct + 1) + cell] + slot;
    a.d.sorted_atom[pos] = i;
    a.d.sorted_q[pos * 3 + 0] = a.q[row * 3 + 0];
    a.d.sorted_q[pos * 3 + 1] = a.q[row * 3 + 1];
    a.d.sorted_q[pos * 3 + 2] = a.q[row * 3 + 2];
}

// S:L3 predicate, explicit IEEE round-to-nearest operations in the stated order
__device__ __forceinline__ bool within_cutoff(const double qi[3], const double *__restrict__ qj, const NlArgs &a, double r2)
{
    double d[3];
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) {
        double dx = __dsub_rn(qj[ax], qi[ax]);
        if (a.periodic) dx = __dsub_rn(dx, __dmul_rn(a.box[ax], round(__ddiv_rn(dx, a.box[ax]))));
        d[ax] = dx;
    }
    double d2 = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
    return d2 < r2;
}

// One CTA per (bead-system, cell).  The atoms of the cell's de-duplicated 3x3x3 stencil are staged in shared memory
// once (index + fp32 position relative to the cell's first atom, CAND_CHUNK at a time); a lane is a home atom and the four
// warps share the candidates, so one broadcast 128-bit shared-memory load serves 32 tests.  The candidates are read from
// HBM/L2 once per cell instead of once per row.  Hits are parked, unsorted, in the row's fixed-stride scratch through a
// shared-memory counter per home atom (integer atomics: the order varies, the fill kernel sorts).
constexpr int CAND_CHUNK = 1024, COUNT_THREADS = 128, HOME_MAX = 128;

// WRAP = false when every periodic axis has at least four cells: home atom and candidate are both stored relative to the same
// reference atom (minimum image), the candidate's cell is at most one cell away from the home cell, so |dx| < 3 cells; when
// |dx| > L/2 the other image is farther than L - 3 L/nc >= one cell width >= r_c: not a neighbour with either image, and the
// per-pair image shift can be left out.
template <bool WRAP>
__global__ void __launch_bounds__(COUNT_THREADS) count_cell_kernel(NlArgs a)
{ pdl_enter();
    __shared__ int sp[CAND_CHUNK];             // candidate: position in the cell-ordered arrays
    __shared__ int cfirst[28], cpre[28];       // first sorted position (relative to the system) and prefix count per stencil cell
    __shared__ int n_st;
    __shared__ double hq[3][HOME_MAX];         // atoms of the home cell (the first HOME_MAX; the rest are read from global)
    __shared__ int hj[HOME_MAX];
    __shared__ int scnt[HOME_MAX];             // hits per home atom so far
    __shared__ float4 sc[CAND_CHUNK];          // candidate: position relative to the cell's reference atom (minimum image, fp32) | atom index
    if (!*a.need) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int sys = blockIdx.x / a.nct, cell = blockIdx.x - sys * a.nct;
    const int *start = a.d.cell_start + (size_t)sys * (a.nct + 1);
    const int h0 = start[cell], nh = start[cell + 1] - h0;
    if (nh == 0) return;                       // uniform: every row belongs to exactly one (non-empty) cell
    const int64_t sbase = (int64_t)sys * a.N;
    // stencil cells: every thread derives the de-duplicated per-axis lists; thread t < n_st loads cell t's range
    {
        int cc[3];
        cc[2] = cell % a.nc[2]; cc[1] = (cell / a.nc[2]) % a.nc[1]; cc[0] = cell / (a.nc[2] * a.nc[1]);
        int lst[3][3], cnt[3];
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) {
            cnt[ax] = 0;
#pragma unroll
            for (int o = -1; o <= 1; ++o) {
                int c = cc[ax] + o;
                if (a.periodic) c = ((c % a.nc[ax]) + a.nc[ax]) % a.nc[ax];
                else if (c < 0 || c >= a.nc[ax]) continue;
                bool dup = false;
                for (int t = 0; t < cnt[ax]; ++t) dup |= (lst[ax][t] == c);
                if (!dup) lst[ax][cnt[ax]++] = c;
            }
        }
        const int ns = cnt[0] * cnt[1] * cnt[2];
        if (tid < ns) {
            const int iz = tid % cnt[2], iy = (tid / cnt[2]) % cnt[1], ix = tid / (cnt[2] * cnt[1]);
            int cx = lst[0][0], cy = lst[1][0], cz = lst[2][0];   // dynamic index into a register array, by selection
#pragma unroll
            for (int t = 1; t < 3; ++t) { if (ix == t) cx = lst[0][t]; if (iy == t) cy = lst[1][t]; if (iz == t) cz = lst[2][t]; }
            const int c = (cx * a.nc[1] + cy) * a.nc[2] + cz;
            cfirst[tid] = start[c];
            cpre[tid + 1] = start[c + 1] - start[c];   // counts; prefix below
        }
        __syncthreads();
        if (tid == 0) {
            int tot = 0;
            cpre[0] = 0;
            for (int k = 0; k < ns; ++k) { const int c = cpre[k + 1]; cpre[k] = tot; tot += c; }
            cpre[ns] = tot;
            n_st = ns;
        }
        for (int t = tid; t < nh; t += COUNT_THREADS) {                   // home atoms
            const int64_t posi = sbase + h0 + t;
            if (t >= HOME_MAX) { a.d.nnz[sbase + a.d.sorted_atom[posi]] = 0; continue; }   // (very full cells: counter in global memory)
            scnt[t] = 0;
            hj[t] = a.d.sorted_atom[posi];
            hq[0][t] = a.d.sorted_q[posi * 3]; hq[1][t] = a.d.sorted_q[posi * 3 + 1]; hq[2][t] = a.d.sorted_q[posi * 3 + 2];
        }
    }
    __syncthreads();
    const int total = cpre[n_st];
    // reference point of the cell: its first atom.  Relative fp32 coordinates are small whatever the absolute ones are.
    const double ref[3] = {a.d.sorted_q[(sbase + h0) * 3], a.d.sorted_q[(sbase + h0) * 3 + 1], a.d.sorted_q[(sbase + h0) * 3 + 2]};
    const float bxf[3] = {a.boxf[0], a.boxf[1], a.boxf[2]};
    const float inf = __int_as_float(0x7f800000);
    const float hbx[3] = {a.periodic ? 0.5f * bxf[0] : inf, a.periodic ? 0.5f * bxf[1] : inf, a.periodic ? 0.5f * bxf[2] : inf};
    const float rc2_hi = a.rc2_hi, rc2_lo = a.rc2_lo;
    for (int base = 0; base < total; base += CAND_CHUNK) {
        const int n = min(CAND_CHUNK, total - base);
        for (int t = tid; t < n; t += COUNT_THREADS) {
            const int idx = base + t;
            int k = 0;
            while (idx >= cpre[k + 1]) ++k;    // <= 27 steps
            const int64_t pos = sbase + cfirst[k] + (idx - cpre[k]);
            sp[t] = (int)(pos - sbase);
            float rel[3];
#pragma unroll
            for (int ax = 0; ax < 3; ++ax) {
                double d = a.d.sorted_q[pos * 3 + ax] - ref[ax];          // once per candidate and cell: fp64 image shift, then fp32
                if (a.periodic) d -= a.box[ax] * rint(d * a.inv_box[ax]);   // (fp32 estimate only: the exact test is within_cutoff)
                rel[ax] = (float)d;
            }
            sc[t] = make_float4(rel[0], rel[1], rel[2], __int_as_float(a.d.sorted_atom[pos]));   // one 128-bit load per test
        }
        __syncthreads();
        // lane = home atom (groups of 32), the four warps share the candidates: one broadcast 128-bit load serves 32 tests.
        // Hits are appended to the row's scratch through a shared-memory counter (their order is free: the fill kernel sorts).
        for (int hg = 0; hg < nh; hg += 32) {
            const int ha = hg + lane;
            const bool act = ha < nh, in_s = ha < HOME_MAX;
            const int64_t posi = sbase + h0 + (act ? ha : 0);
            const int i = !act ? -1 : (in_s ? hj[ha] : a.d.sorted_atom[posi]);
            const int64_t row = sbase + (act ? i : 0);
            int *buf = a.d.hits + row * a.hit_stride;
            float qif[3];
#pragma unroll
            for (int ax = 0; ax < 3; ++ax) {
                double d = ((act && in_s) ? hq[ax][ha] : a.d.sorted_q[posi * 3 + ax]) - ref[ax];
                if (a.periodic) d -= a.box[ax] * rint(d * a.inv_box[ax]);   // (fp32 estimate only: the exact test is within_cutoff)
                qif[ax] = (float)d;
            }
            // 32 of this warp's candidates at a time (s = sb + 4 k).  The tests only set a bit per candidate -- clear hit, or inside
            // the band; nearly every candidate is a hit for SOME lane of the warp, so a branch per candidate would send the whole warp
            // through the append path every time.  The set bits (13 % of a lane's candidates) are handled after the block.
            constexpr int NWARP = COUNT_THREADS / 32;
            for (int sb = warp; sb < n; sb += 32 * NWARP) {
                unsigned hitm = 0u, bandm = 0u;
#pragma unroll
                for (int k = 0; k < 32; ++k) {
                    const int s0 = sb + k * NWARP;
                    const float4 cj = sc[s0 < n ? s0 : n - 1];
                    float d2 = 0.f;
#pragma unroll
                    for (int ax = 0; ax < 3; ++ax) {
                        float dx = (ax == 0 ? cj.x : (ax == 1 ? cj.y : cj.z)) - qif[ax];
                        if (WRAP) {
                            float sh = (dx > hbx[ax]) ? bxf[ax] : 0.f;      // selects, not branches (hbx = +inf when not periodic)
                            sh = (dx < -hbx[ax]) ? -bxf[ax] : sh;
                            dx -= sh;
                        }
                        d2 = fmaf(dx, dx, d2);
                    }
                    const bool cand = (s0 < n) && (__float_as_int(cj.w) != i);
                    d2 = cand ? d2 : inf;        // not a candidate: neither a hit nor in the band
                    // (predicated ORs: written as selects, the two masks cost more than the branch they replace)
                    asm("{\n\t.reg .pred ph, pb;\n\t"
                        "setp.lt.f32 ph, %2, %3;\n\t"
                        "setp.le.and.f32 pb, %2, %4, !ph;\n\t"
                        "@ph or.b32 %0, %0, %5;\n\t"
                        "@pb or.b32 %1, %1, %5;\n\t}"
                        : "+r"(hitm), "+r"(bandm) : "f"(d2), "f"(rc2_lo), "f"(rc2_hi), "r"(1u << k));
                }
                if (!act) { hitm = 0u; bandm = 0u; }
                while (bandm) {                  // in the band (about 0.2 % of the candidates): fp64 positions, exact S:L3 sequence
                    const int k = __ffs(bandm) - 1;
                    bandm &= bandm - 1;
                    const double qi[3] = {in_s ? hq[0][ha] : a.d.sorted_q[posi * 3], in_s ? hq[1][ha] : a.d.sorted_q[posi * 3 + 1],
                                          in_s ? hq[2][ha] : a.d.sorted_q[posi * 3 + 2]};
                    if (within_cutoff(qi, a.d.sorted_q + (sbase + sp[sb + k * NWARP]) * 3, a, a.rl2)) hitm |= 1u << k;
                }
                if (hitm) {
                    int idx = in_s ? atomicAdd(&scnt[ha], __popc(hitm)) : atomicAdd(&a.d.nnz[row], __popc(hitm));
                    while (hitm) {
                        const int k = __ffs(hitm) - 1;
                        hitm &= hitm - 1;
                        if (idx < a.hit_stride) buf[idx] = __float_as_int(sc[sb + k * NWARP].w);
                        ++idx;
                    }
                }
            }
        }
        __syncthreads();
    }
    for (int t = tid; t < nh; t += COUNT_THREADS) {                       // counts; a row with more hits than its scratch holds is an error
        const int64_t row = sbase + ((t < HOME_MAX) ? hj[t] : a.d.sorted_atom[sbase + h0 + t]);
        int cnt = (t < HOME_MAX) ? scnt[t] : a.d.nnz[row];
        if (cnt > a.hit_stride) { atomicOr(a.err, PIMD_FLAG_PAIRS); cnt = a.hit_stride; }
        a.d.ncand[row] = cnt;
    }
}

// candidates of a row -> ascending j, in place: the row's candidates set bits in a per-warp bitmask over the atoms of the
// bead-system (shared memory, N/32 words) and the set bits are written back in order.  N <= 32768 (checked by pimd_create).
__global__ void __launch_bounds__(256) sort_candidates_kernel(NlArgs a, int nw)
{ pdl_enter();
    extern __shared__ unsigned smask[];       // [8][nw] bitmask, [8][nw] set bits in the words before, [8][hit_stride] sorted row
    if (!*a.need) return;
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * 8 + w;
    if (row >= a.rows) return;
    unsigned *mk = smask + (size_t)w * nw, *pre = smask + (size_t)(8 + w) * nw;
    int *stage = (int *)(smask + (size_t)16 * nw) + (size_t)w * a.hit_stride;
    const int n = a.d.ncand[row];
    int *hits = a.d.hits + row * a.hit_stride;
    for (int t = lane; t < nw; t += 32) mk[t] = 0u;
    __syncwarp();
    for (int e = lane; e < n; e += 32) {
        const int j = hits[e];
        atomicOr(&mk[j >> 5], 1u << (j & 31));
    }
    __syncwarp();
    const int wpl = (nw + 31) >> 5, w0 = lane * wpl, w1 = min(w0 + wpl, nw);
    int cnt = 0;
    for (int t = w0; t < w1; ++t) cnt += __popc(mk[t]);
    int inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += v;
    }
    int run = inc - cnt;
    for (int t = w0; t < w1; ++t) { pre[t] = (unsigned)run; run += __popc(mk[t]); }
    __syncwarp();
    // a candidate is stored as j (15 bits) | image shift of the pair at the reference positions, five bits per axis (biased by 16:
    // positions are never wrapped, S:L2, so the shift can be several box lengths) | bit 30 if a shift does not fit (the filter
    // then takes the exact path).  The shift cannot change while the list is in use in a way that matters: a pair whose
    // minimum image flips is at least r_cut apart with either image (box >= 2 (r_cut + skin)).
    // Every lane packs the candidates it holds; a candidate's place in the row is the number of set bits below it.  The row is
    // put in order in shared memory and written back in place.
    const int64_t sbase = (row / a.N) * a.N;
    const double qi[3] = {a.q[row * 3], a.q[row * 3 + 1], a.q[row * 3 + 2]};
    for (int e = lane; e < n; e += 32) {
        const int j = hits[e];
        int packed = j;
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) {
            int sh = 0;
            if (a.periodic) sh = (int)rint((a.q[(sbase + j) * 3 + ax] - qi[ax]) / a.box[ax]);
            if (sh < -16 || sh > 15) { packed |= 1 << 30; sh = 0; }
            packed |= (sh + 16) << (15 + 5 * ax);
        }
        stage[(int)pre[j >> 5] + __popc(mk[j >> 5] & ((1u << (j & 31)) - 1u))] = packed;
    }
    __syncwarp();
    for (int e = lane; e < n; e += 32) hits[e] = stage[e];
}

// every step: the exact list from the sorted candidates.  One warp per row; a lane tests candidates e = lane, lane + 32, ...:
// an fp32 estimate from the fp32 copy of the positions and the stored image shift settles everything outside a 2e-4 band
// around r_c^2, the fp64 predicate of S:L3 decides inside it; the ballots are kept as the row's hit mask.
constexpr int MASK_WORDS = PIMD_MAX_NBR / 32;
__global__ void __launch_bounds__(256) filter_count_kernel(NlArgs a)
{ pdl_enter();
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * 8 + w;
    if (row >= a.rows) return;
    const int n = a.d.ncand[row];
    const int *cand = a.d.hits + row * a.hit_stride;
    const int64_t sbase = (row / a.N) * a.N;
    const float4 qi = a.d.q32[row];
    const float lo = (float)(a.rc2 * (1.0 - 2e-4)), hi = (float)(a.rc2 * (1.0 + 2e-4));   // fp32 absolute coordinates: error << band
    int cnt = 0;
    for (int e0 = 0; e0 < n; e0 += 32) {
        const int e = e0 + lane;
        bool hit = false;
        if (e < n) {
            const int pk = cand[e], j = pk & 0x7FFF;
            const float4 qj = __ldg(a.d.q32 + sbase + j);
            const float dx = (qj.x - qi.x) - (float)(((pk >> 15) & 31) - 16) * a.boxf[0];
            const float dy = (qj.y - qi.y) - (float)(((pk >> 20) & 31) - 16) * a.boxf[1];
            const float dz = (qj.z - qi.z) - (float)(((pk >> 25) & 31) - 16) * a.boxf[2];
            const float d2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
            hit = d2 < lo && !(pk & (1 << 30));
            if ((!hit && d2 <= hi) || (pk & (1 << 30))) {   // in the band (or shift not stored): the exact fp64 operation sequence of S:L3 decides
                const double qid[3] = {a.q[row * 3], a.q[row * 3 + 1], a.q[row * 3 + 2]};
                hit = within_cutoff(qid, a.q + (sbase + j) * 3, a, a.rc2);
            }
        }
        const unsigned m = __ballot_sync(0xffffffffu, hit);
        if (lane == 0) a.d.hitmask[row * MASK_WORDS + (e0 >> 5)] = m;
        cnt += __popc(m);
    }
    if (lane == 0) a.d.nnz[row] = cnt;
}

// the list's total: checked against the capacity, stored behind the last row
__device__ __forceinline__ void store_total(const NlArgs &a, long long total)
{
    if (total > a.d.pair_cap || total > 2147483647LL) {
        atomicOr(a.err, PIMD_FLAG_PAIRS);
        total = 0;   // downstream kernels see an empty list instead of reading out of bounds
    }
    a.d.row_ptr[a.rows] = (int)total;
}

// row_ptr: exclusive scan over rows in two kernels (1024 rows per block; block offsets), the offsets are added by the fill kernel
// of the list (row_start below).  Up to 1024 rows the first kernel is the whole scan.
__global__ void __launch_bounds__(1024) scan_rows_local_kernel(NlArgs a)
{ pdl_enter();
    __shared__ int tot;
    int64_t row = (int64_t)blockIdx.x * 1024 + threadIdx.x;
    int v = (row < a.rows) ? a.d.nnz[row] : 0;
    int ex = block_exclusive_scan(v, &tot);
    if (row < a.rows) a.d.row_ptr[row] = ex;
    if (threadIdx.x == 0) {
        if (gridDim.x == 1) { a.d.block_sums[0] = 0; store_total(a, tot); }
        else a.d.block_sums[blockIdx.x] = tot;
    }
}

// start of the row in the pair list: block-local prefix + block offset, stored as the final row_ptr by the row's warp (no other
// warp reads this entry before the kernel ends)
__device__ __forceinline__ int64_t row_start(const NlArgs &a, int64_t row, int lane)
{
    int base = 0;
    if (lane == 0) {
        base = a.d.row_ptr[row] + a.d.block_sums[row >> 10];
        a.d.row_ptr[row] = base;
    }
    return (int64_t)__shfl_sync(0xffffffffu, base, 0);
}

__global__ void __launch_bounds__(1024) scan_block_sums_kernel(NlArgs a, int nblocks)
{ pdl_enter();
    __shared__ int tot;
    long long carry = 0;
    for (int base = 0; base < nblocks; base += 1024) {
        int b = base + threadIdx.x;
        int v = (b < nblocks) ? a.d.block_sums[b] : 0;
        int ex = block_exclusive_scan(v, &tot);
        if (b < nblocks) a.d.block_sums[b] = (int)(carry + ex);
        carry += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) store_total(a, carry);
}

// Geometry of a pair for the tensor-core pair pipeline (gfn_pair_pipe.cu, role P), written where the pair is emitted: r_j - r_i as
// the fp64 difference with the minimum image, then fp32 (S:G1: the value role P would otherwise form itself behind the dependent
// load chain pair -> row, column -> positions), and the kind of the row's segment inside the pair's 32-pair granule
// (0 whole row, 1 began in an earlier granule, 2 continues into a later one).
__device__ __forceinline__ void store_pair_geometry(const NlArgs &a, const double (&qi)[3], int64_t sbase, int j, int64_t rs, int n, int64_t pos)
{
    float f[3];
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) {
        double dx = a.q[(sbase + j) * 3 + ax] - qi[ax];
        if (a.periodic) dx = dx - a.box[ax] * rint(dx * a.inv_box[ax]);
        f[ax] = (float)dx;
    }
    const int64_t g0 = pos & ~(int64_t)31;
    const int kind = (rs >= g0 && rs + n <= g0 + 32) ? 0 : ((rs < g0) ? 1 : 2);
    a.d.dvec[pos] = make_float4(f[0], f[1], f[2], __int_as_float(kind));
}

// CSR fill with ascending rows and no sort: the row's hits set bits in a per-warp bitmask over the atoms of the bead-system
// (shared memory, N/32 words); a hit's place in the row is the number of set bits below it (per-word prefix counts, then one
// popc), so every hit is stored by the lane that holds it -- no serial walk over the set bits.  N <= 32768 (pimd_create).
__global__ void __launch_bounds__(256) fill_bitmask_kernel(NlArgs a, int nw)
{ pdl_enter();
    extern __shared__ unsigned smask[];       // [8][nw] bitmask, then [8][nw] set bits in the words before
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * 8 + w;
    if (row >= a.rows) return;
    const int64_t base = row_start(a, row, lane);
    if (a.d.row_ptr[a.rows] == 0) return;     // empty or overflowed list
    unsigned *mk = smask + (size_t)w * nw, *pre = smask + (size_t)(8 + w) * nw;
    const int n = a.d.nnz[row];
    const int *hits = a.d.hits + row * a.hit_stride;
    for (int t = lane; t < nw; t += 32) mk[t] = 0u;
    __syncwarp();
    for (int e = lane; e < n; e += 32) {
        const int j = hits[e];
        atomicOr(&mk[j >> 5], 1u << (j & 31));
    }
    __syncwarp();
    const int wpl = (nw + 31) >> 5, w0 = lane * wpl, w1 = min(w0 + wpl, nw);
    int cnt = 0;
    for (int t = w0; t < w1; ++t) cnt += __popc(mk[t]);
    int inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += v;
    }
    int run = inc - cnt;
    for (int t = w0; t < w1; ++t) { pre[t] = (unsigned)run; run += __popc(mk[t]); }
    __syncwarp();
    int *col = a.d.col + base, *prow = a.d.pair_row + base;
    const int64_t sbase = (row / a.N) * a.N;
    const double qi[3] = {a.q[row * 3], a.q[row * 3 + 1], a.q[row * 3 + 2]};
    for (int e = lane; e < n; e += 32) {
        const int j = hits[e];
        const int pos = (int)pre[j >> 5] + __popc(mk[j >> 5] & ((1u << (j & 31)) - 1u));
        col[pos] = j;
        prow[e] = (int)row;                   // coalesced
    }
    if (a.d.dvec) {                           // second walk, in list order: coalesced 16-byte stores, ascending j
        __syncwarp();
        for (int e = lane; e < n; e += 32) store_pair_geometry(a, qi, sbase, col[e], base, n, base + e);
    }
}

// ---- small open clusters (one cell per bead-system, N <= BRUTE_MAX_N: the FAD configs): the cell machinery above is seven launches
// for a list that one thread per row writes directly.  Thread = row i; j runs over the bead-system in ascending order with the
// exact S:L3 predicate (the definition itself: S:L1), so the rows are ascending by construction.
//   SINGLE: rows <= 1024, one block is the whole list: count, block scan, fill in one launch.
//   else  : brute_count_kernel (count + block-local scan + block sums), scan_block_sums_kernel, brute_fill_kernel.
constexpr int BRUTE_MAX_N = 128;

__device__ __forceinline__ int brute_row(const NlArgs &a, int64_t row, int64_t base, bool write)
{
    const int64_t sbase = (row / a.N) * a.N;
    const int i = (int)(row - sbase);
    const double qi[3] = {a.q[row * 3], a.q[row * 3 + 1], a.q[row * 3 + 2]};
    int n = 0;
    for (int j = 0; j < a.N; ++j) {
        if (j == i || !within_cutoff(qi, a.q + (sbase + j) * 3, a, a.rc2)) continue;
        if (write) { a.d.col[base + n] = j; a.d.pair_row[base + n] = (int)row; }
        ++n;
    }
    return n;
}

__device__ __forceinline__ void brute_geometry(const NlArgs &a, int64_t row, int64_t base, int n)
{
    if (!a.d.dvec) return;
    const int64_t sbase = (row / a.N) * a.N;
    const double qi[3] = {a.q[row * 3], a.q[row * 3 + 1], a.q[row * 3 + 2]};
    for (int e = 0; e < n; ++e) store_pair_geometry(a, qi, sbase, a.d.col[base + e], base, n, base + e);
}

template <bool SINGLE>
__global__ void __launch_bounds__(1024) brute_count_kernel(NlArgs a)
{ pdl_enter();
    __shared__ int tot;
    const int64_t row = (int64_t)blockIdx.x * 1024 + threadIdx.x;
    if (row == 0) a.need_w[1] += 1;            // rebuild counter (pimd_nlist_rebuilds)
    const int n = (row < a.rows) ? brute_row(a, row, 0, false) : 0;
    const int ex = block_exclusive_scan(n, &tot);
    if (!SINGLE) {
        if (row < a.rows) { a.d.nnz[row] = n; a.d.row_ptr[row] = ex; }
        if (threadIdx.x == 0) a.d.block_sums[blockIdx.x] = tot;
        return;
    }
    // the whole list is this block's
    const bool fits = (long long)tot <= a.d.pair_cap;
    if (threadIdx.x == 0) { a.d.block_sums[0] = 0; store_total(a, tot); }
    if (row < a.rows) {
        a.d.nnz[row] = n;
        a.d.row_ptr[row] = fits ? ex : 0;
        if (fits && n > 0) { brute_row(a, row, ex, true); brute_geometry(a, row, ex, n); }
    }
}

__global__ void __launch_bounds__(256) brute_fill_kernel(NlArgs a)
{ pdl_enter();
    const int64_t row = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (row >= a.rows) return;
    const int base = a.d.row_ptr[row] + a.d.block_sums[row >> 10];
    a.d.row_ptr[row] = base;
    if (a.d.row_ptr[a.rows] == 0) return;      // empty or overflowed list
    const int n = a.d.nnz[row];
    if (n > 0) { brute_row(a, row, base, true); brute_geometry(a, row, base, n); }
}

// CSR fill: the row's hit mask selects from its sorted candidates, so the rows come out in ascending j
__global__ void __launch_bounds__(256) filter_fill_kernel(NlArgs a)
{ pdl_enter();
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * 8 + w;
    if (blockIdx.x == 0 && threadIdx.x == 0) *a.need_w = 0;   // the candidate lists are current; the next check may raise the flag again
    if (row >= a.rows) return;
    int64_t base = row_start(a, row, lane);
    if (a.d.row_ptr[a.rows] == 0) return;     // empty or overflowed list
    const int n = a.d.ncand[row];
    const int *cand = a.d.hits + row * a.hit_stride;
    const int64_t rs = base, sbase = (row / a.N) * a.N;
    const int nn = a.d.nnz[row];
    const double qi[3] = {a.q[row * 3], a.q[row * 3 + 1], a.q[row * 3 + 2]};
    for (int e0 = 0; e0 < n; e0 += 32) {
        const unsigned m = a.d.hitmask[row * MASK_WORDS + (e0 >> 5)];
        const int e = e0 + lane;
        if ((m >> lane) & 1u) {
            const int pos = __popc(m & ((1u << lane) - 1u));
            const int j = cand[e] & 0x7FFF;
            a.d.col[base + pos] = j;
            a.d.pair_row[base + pos] = (int)row;
            if (a.d.dvec) store_pair_geometry(a, qi, sbase, j, rs, nn, base + pos);
        }
        base += __popc(m);
    }
}

}  // namespace

__global__ void set_flag_kernel(int *f, int v) { pdl_enter(); *f = v; }

int pimd_launch_nlist(pimd_ctx *c)
{
    NlArgs a;
    a.N = c->N; a.nsys = c->R * c->P; a.periodic = c->periodic; a.rows = c->rows;
    for (int k = 0; k < 3; ++k) { a.box[k] = c->box[k]; a.inv_box[k] = c->periodic ? 1.0 / c->box[k] : 0.0; a.nc[k] = c->nl.ncell[k]; }
    a.rc2 = (double)c->net.r_cut * (double)c->net.r_cut;
    const double rl = (double)c->net.r_cut + c->nl.skin;
    a.rl2 = rl * rl;
    a.skin_half2 = 0.25 * c->nl.skin * c->nl.skin;
    a.nct = c->nl.ncell_tot; a.q = c->q; a.d = c->nl; a.err = c->err;
    a.need = c->nl.need; a.need_w = c->nl.need;
    a.rc2_lo = (float)(a.rl2 * (1.0 - 1e-3)); a.rc2_hi = (float)(a.rl2 * (1.0 + 1e-3));
    for (int k = 0; k < 3; ++k) { a.boxf[k] = (float)c->box[k]; a.inv_boxf[k] = c->periodic ? (float)(1.0 / c->box[k]) : 0.f; }
    a.hit_stride = c->nl.hit_stride;
    const int64_t rows = c->rows;
    const unsigned gthr = (unsigned)((rows + 255) / 256), gwarp = (unsigned)((rows + 7) / 8);
    const int nblk = (int)((rows + 1023) / 1024);
    const int nw = (c->N + 31) / 32;
    const bool wrap = a.periodic && (a.nc[0] < 4 || a.nc[1] < 4 || a.nc[2] < 4);
    if (c->nl.skin == 0.0 && a.nct == 1 && c->N <= BRUTE_MAX_N) {
        // small open clusters: one thread per row, one launch up to 1024 rows, three above
        if (nblk == 1) {
            pimd_launch(brute_count_kernel<true>, 1, 1024, 0, c->stream, a);
            c->launches += 1;
        } else {
            pimd_launch(brute_count_kernel<false>, nblk, 1024, 0, c->stream, a);
            pimd_launch(scan_block_sums_kernel, 1, 1024, 0, c->stream, a, nblk);
            pimd_launch(brute_fill_kernel, gthr, 256, 0, c->stream, a);
            c->launches += 3;
        }
        PIMD_CUDA_CHECK(cudaGetLastError());
        return 0;
    }
    if (c->nl.skin == 0.0) {
        // no reuse: the cell-list pass at r_cut IS the list of this step (count -> scan -> fill through the bitmask, ascending j)
        a.d.nnz = a.d.ncand;           // the count kernel's output is the row length
        if (!c->nl_flag_up) {             // nothing lowers the flag on this path: raised once (after a change of the skin)
            pimd_launch(set_flag_kernel, 1, 1, 0, c->stream, c->nl.need, 1);
            c->nl_flag_up = true;
            c->launches++;
        }
        PIMD_CUDA_CHECK(cudaMemsetAsync(c->nl.cell_count, 0, sizeof(int) * (size_t)a.nsys * a.nct, c->stream));
        pimd_launch(bin_kernel, gthr, 256, 0, c->stream, a);
        pimd_launch(scan_cells_kernel, a.nsys, 256, 0, c->stream, a);
        pimd_launch(scatter_kernel, gthr, 256, 0, c->stream, a);
        if (wrap) pimd_launch(count_cell_kernel<true>, (unsigned)(a.nsys * a.nct), COUNT_THREADS, 0, c->stream, a);
        else pimd_launch(count_cell_kernel<false>, (unsigned)(a.nsys * a.nct), COUNT_THREADS, 0, c->stream, a);
        pimd_launch(scan_rows_local_kernel, nblk, 1024, 0, c->stream, a);
        if (nblk > 1) pimd_launch(scan_block_sums_kernel, 1, 1024, 0, c->stream, a, nblk);
        const size_t fill_smem = (size_t)16 * nw * sizeof(unsigned);
        if (fill_smem > 48 * 1024 && !(c->attr_done & ATTR_FILL)) {   // (the first step of a context is never captured)
            PIMD_CUDA_CHECK(cudaFuncSetAttribute(fill_bitmask_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024));
            c->attr_done |= ATTR_FILL;
        }
        pimd_launch(fill_bitmask_kernel, gwarp, 256, fill_smem, c->stream, a, nw);
        c->launches += 6 + (nblk > 1);
        PIMD_CUDA_CHECK(cudaGetLastError());
        return 0;
    }
    // candidate lists (r_cut + skin): rebuilt only when the flag is up; these kernels return at once otherwise
    pimd_launch(verlet_check_kernel, gthr, 256, 0, c->stream, a);
    PIMD_CUDA_CHECK(cudaMemsetAsync(c->nl.cell_count, 0, sizeof(int) * (size_t)a.nsys * a.nct, c->stream));
    pimd_launch(bin_kernel, gthr, 256, 0, c->stream, a);
    pimd_launch(scan_cells_kernel, a.nsys, 256, 0, c->stream, a);
    pimd_launch(scatter_kernel, gthr, 256, 0, c->stream, a);
    if (wrap) pimd_launch(count_cell_kernel<true>, (unsigned)(a.nsys * a.nct), COUNT_THREADS, 0, c->stream, a);
    else pimd_launch(count_cell_kernel<false>, (unsigned)(a.nsys * a.nct), COUNT_THREADS, 0, c->stream, a);
    {
        const size_t sort_smem = ((size_t)16 * nw + (size_t)8 * c->nl.hit_stride) * sizeof(unsigned);
        if (sort_smem > 48 * 1024 && !(c->attr_done & ATTR_SORT)) {
            PIMD_CUDA_CHECK(cudaFuncSetAttribute(sort_candidates_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
            c->attr_done |= ATTR_SORT;
        }
        pimd_launch(sort_candidates_kernel, gwarp, 256, sort_smem, c->stream, a, nw);
    }
    // exact list of this step, filtered from the candidates
    pimd_launch(filter_count_kernel, gwarp, 256, 0, c->stream, a);
    pimd_launch(scan_rows_local_kernel, nblk, 1024, 0, c->stream, a);
    if (nblk > 1) pimd_launch(scan_block_sums_kernel, 1, 1024, 0, c->stream, a, nblk);
    pimd_launch(filter_fill_kernel, gwarp, 256, 0, c->stream, a);
    c->nl_flag_up = false;               // (the fill kernel lowers the flag)
    c->launches += 9 + (nblk > 1);
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}

// raises the rebuild flag (new positions from outside, new skin)
int pimd_launch_nlist_invalidate(pimd_ctx *c)
{
    if (c->kind != 0) return 0;
    pimd_launch(set_flag_kernel, 1, 1, 0, c->stream, c->nl.need, 1);
    c->nl_flag_up = true;
    c->launches++;
    PIMD_CUDA_CHECK(cudaGetLastError());
    return 0;
}
