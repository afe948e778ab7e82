// dtw_kernel.cuh -- sm_100a kernel of the Step-3 scoring path: classic DTW (eq. 1,
// PAPER.md:123-127) between the prototype Z and each cycle x_k, the length |pi| of the optimal alignment path, and
// the similarity score d_score = DTW / |pi| (Def. 8 / eq. 8).
//
//   r_ij = D_ij + min(r_{i-1,j-1}, r_{i-1,j}, r_{i,j-1}),   r_00 = 0, r_i0 = r_0j = +inf          (eq. 5 with gamma = 0)
//   len_ij = 1 + len of the FIRST of (diagonal, up, left) that attains the minimum                 (C20)
//
// Natural units (no scaling), plain float32 with one rounding per operation and no fused multiply-add, so that the
// integer |pi| -- decided by float comparisons -- can be compared bit for bit with a float32 mirror of the same
// recurrence:  D = sum_c fl(fl(x_c - z_c)^2) (c ascending),  r = fl(D + min).
//
// Same wavefront as the Soft-DTW forward kernel (sdtw_kernels.cuh): a work item is one strip of 32 x W columns of one
// pair swept by one warp, lane l on rows 2(s-l), 2(s-l)+1 at step s; (r, len) of a lane's last column goes to the next
// lane by shuffle and to the next strip through a sentinel-preset global column polled one chunk ahead.  No special
// functions: the bound is the FP32/ALU issue rate.  Two layouts.  COLUMNS (FW = 8): items are handed out strip-major from
// one atomic counter to independent warps (every item's producer was handed out earlier, so a waiting warp never blocks
// the warp it waits for) and every strip keeps a boundary column.  RINGS (FW = 32, chosen when the problem has more
// strips than resident warps, d <= 2): the forward kernel's schedule -- units of 32 adjacent strips popped group-major by
// a CTA whose warps serve a rolling stream of strips -- with the boundary values travelling inside a unit through
// per-warp rings (as in the forward-only Soft-DTW sweep; an entry carries (r, len) of two rows as four tagged 64-bit
// words); only the last strip of a unit keeps a full column.  cfg 5: 56.7 -> 1.9 GB of workspace, 326 -> 352 ms.
#pragma once
#include "sdtw_kernels.cuh"

namespace sdtw {

// warps per CTA: 8 independent warps in the column layout; a CTA-full of 32 (= strips per unit) in the ring layout, which
// exists at d <= 2 only (the kernel fits 64 registers there)
constexpr int DTW_WARPS = 8;
constexpr int DTW_RING_WARPS = 32;
#ifndef SDTW_DTW_RING_CHUNKS
#define SDTW_DTW_RING_CHUNKS 8
#endif
// ring of the DTW kernels: 32 bytes per entry, so half as many chunks as the Soft-DTW ring keep the rings of all resident
// warps (148 x 32 x 8 KB = 39 MB) inside the L2 (with 16 chunks the ring traffic, 96 GB on cfg 5, went through HBM)
constexpr int DTW_RING_CHUNKS = SDTW_DTW_RING_CHUNKS;
constexpr int DTW_RING_ENTRIES = DTW_RING_CHUNKS * CH;
static_assert((DTW_RING_ENTRIES & (DTW_RING_ENTRIES - 1)) == 0, "ring size is a power of two");
#ifndef SDTW_DTW_W
#define SDTW_DTW_W 4
#endif
// columns per thread of the DTW kernels: wider than the Soft-DTW tile (fewer shuffles / boundary words per cell; the cell
// is cheap and has no special functions to hide); narrower at many channels, where z[DW][D] would spill
template <int D> __host__ __device__ constexpr int dtw_w() { return D <= 2 ? SDTW_DTW_W : 4; }
constexpr unsigned F_INF = 0x7f800000u;

struct DtwParams {
    const float* Z;       // [m][D] natural units
    const float* X;       // [sum n][D]
    const PairMeta* pm;   // schedule order; vs_off / vs_stride in 32-bit words, 2 words (r, len) per row
    unsigned* counter;    // work queue (units)
    unsigned* VS;         // strip-boundary columns: word 2 row = r bits, word 2 row + 1 = len
    unsigned long long* ring;   // [CTA][warp position][RING_ENTRIES][4]: (r, len) of a row pair, each word | tag << 32; or null
    unsigned* ring_prog;        // [CTA][warp position] entries of the left neighbour's ring this warp has consumed
    float* out_dtw;       // [N] caller order (may be null): DTW, or the Sub-DTW value
    int* out_len;         // [N] (may be null): |pi|, or a* (Sub-DTW)
    float* out_score;     // [N] (may be null): DTW / |pi| (not written by the Sub-DTW variant)
    int* out_b;           // [N] (may be null): b* (Sub-DTW only)
    int m, N, NS;
    unsigned num_items;
};

struct RL { float r; float l; };   // l: path length / start row kept as a float (exact below 2^24): its +1 then runs on the FMA pipe, not the ALU pipe that bounds this kernel

__device__ __forceinline__ uint4 ld_relaxed_u4(const unsigned* p) {
    uint4 v;
    asm volatile("ld.relaxed.gpu.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_u4(unsigned* p, uint4 v) {
    asm volatile("st.relaxed.gpu.global.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

template <int D> __host__ __device__ constexpr int dtw_smem_floats() { return 2 * XWIN * D + 2 * 4 * 32; }

// one cell: (rd, ld) diagonal, (ru, lu) up [in: old row value of this column; out: this cell], (rl, ll) left [in/out]
// SUB (Sub-DTW, eq. 2): the integer carried with the minimum is the path's first row (copied), not its length (+1)
template <int D, bool SUB>
__device__ __forceinline__ void dtw_cell(const XRow<D>& x, const float (&z)[D], float& rd, float& ld, float& ru, float& lu,
                                         float& rl, float& ll) {
    float t = __fsub_rn(x.c[0], z[0]);
    float dist = __fmul_rn(t, t);
#pragma unroll
    for (int c = 1; c < D; ++c) { t = __fsub_rn(x.c[c], z[c]); dist = __fadd_rn(dist, __fmul_rn(t, t)); }
    const float mn = fminf(fminf(rd, ru), rl);
    float lsel;                            // first of (diagonal, up, left) that attains the minimum; branch-free
    asm("{\n\t.reg .pred p, q;\n\t.reg .f32 t;\n\t"
        "setp.eq.f32 p, %1, %2;\n\tsetp.eq.f32 q, %3, %2;\n\t"
        "selp.f32 t, %4, %5, q;\n\tselp.f32 %0, %6, t, p;\n\t}"
        : "=f"(lsel) : "f"(rd), "f"(mn), "f"(ru), "f"(lu), "f"(ll), "f"(ld));
    const float l1 = SUB ? lsel : __fadd_rn(lsel, 1.0f);
    const float rn = __fadd_rn(dist, mn);
    rd = ru; ld = lu;                      // this column's old row value is the next column's diagonal
    ru = rn; lu = l1;
    rl = rn; ll = l1;
}

// SUB = false: eq. 1 / eq. 8 (complete paths).  SUB = true: eq. 2, the rows (the series of
// X_concat) have free ends: r_i0 = 0 for every i, value = min_i r_im, b* = the smallest such i, a* = the path's first row.
template <int D, bool SUB, int FW>
__global__ void __launch_bounds__(FW * 32) dtw_kernel(const DtwParams p) {
    constexpr int W = dtw_w<D>();                                    // shadows sdtw::W inside this kernel
    constexpr bool RINGS = (FW == DTW_RING_WARPS);
    extern __shared__ __align__(16) float smem[];
    __shared__ RollCtl ctl;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float* xs0 = smem + warp * dtw_smem_floats<D>();                 // [2][XWIN][D]
    uint4* vin_s = reinterpret_cast<uint4*>(xs0 + 2 * XWIN * D);     // [CH] (r, len) of the left strip for lane 0's two rows
    uint4* vout_s = vin_s + 32;                                      // [CH] (r, len) of lane 31's last column
    const int m = p.m;
    const float INF = __uint_as_float(F_INF);
    constexpr int US = FW;                                            // RINGS: strips per unit
    const int NG = (p.NS + US - 1) / US, NU = NG * p.N;              // RINGS: units per pair, units
    const int mypos = (warp & 3) * (FW / 4) + (warp >> 2);           // consecutive positions share a scheduler
    if (threadIdx.x < 32) { ctl.seen[threadIdx.x] = 0; if (threadIdx.x == 0) { ctl.popped = 0; ctl.lock = 0; } }
    __syncthreads();

    int base = 0;
    unsigned in_q = 0, out_q = 0;                          // ring entries consumed from the left / produced, all strips so far
    for (int k = 0;; ++k) {
        int J, ps, g = 0, S = 1, sidx = 0;
        if constexpr (RINGS) {
            const int u = pop_unit<FW>(ctl, p.counter, k, NU, warp, lane);
            if (u >= NU) break;
            g = u / p.N; ps = u - g * p.N;                   // group-major: every pair's unit g before any unit g + 1
            S = min(US, p.NS - g * US);
            sidx = (mypos - base + FW) % FW;
            base = (base + S) % FW;
            if (sidx >= S) continue;
            J = g * US + sidx;
        } else {
            unsigned q = 0;
            if (lane == 0) q = atomicAdd(p.counter, 1u);
            q = __shfl_sync(FULL, q, 0);
            if (q >= p.num_items) break;
            J = q / p.N; ps = q - J * p.N;                   // strip-major: every pair's strip J before any strip J + 1
        }
        const PairMeta pm = p.pm[ps];
        const int n = pm.n, C = pm.C;
        const int j0 = (J * 32 + lane) * W;
        constexpr bool rings = RINGS;
        const bool in_ring = rings && sidx > 0, out_ring = rings && sidx + 1 < S;
        const bool out_none = rings && !out_ring && J == p.NS - 1;
        const long long col = rings ? (out_ring ? 0 : g) : J;
        unsigned* VSme = p.VS + pm.vs_off + col * pm.vs_stride + 2 * VS_PAD;   // word 2 row
        const unsigned* VSprev = rings ? p.VS + pm.vs_off + (long long)(g - 1) * pm.vs_stride + 2 * VS_PAD : VSme - pm.vs_stride;
        auto ring_of = [&](const int q) { return p.ring + ((size_t)blockIdx.x * FW + q) * (DTW_RING_ENTRIES * 4); };
        auto prog_of = [&](const int q) { return p.ring_prog + (size_t)blockIdx.x * FW + q; };

        float z[W][D], ru[W], lu[W];
#pragma unroll
        for (int w = 0; w < W; ++w) {
            const int j = j0 + w;
#pragma unroll
            for (int c = 0; c < D; ++c) z[w][c] = (j < m) ? __ldg(p.Z + (long long)j * D + c) : 0.f;
            ru[w] = INF; lu[w] = 0.f;                          // virtual row 0: r_0j = +inf
        }
        RL oA{INF, 0.f}, oB{INF, 0.f};                           // this lane's last column, rows 2(s-l) and 2(s-l)+1
        RL dprev{(J == 0 && lane == 0) ? 0.f : INF, 0.f};      // diagonal of the first column's upper row; r_00 = 0
        const float* xs_lane = xs0;
        const bool last_strip = (J == p.NS - 1);
        float best = INF, best_a = 0.f; int best_b = 0;        // Sub-DTW: running min over rows of r in column m - 1
        auto track = [&](const int i) {
#pragma unroll
            for (int w = 0; w < W; ++w)
                if (j0 + w == m - 1 && ru[w] < best) { best = ru[w]; best_a = lu[w]; best_b = i; }
        };

        auto step = [&](const int c, const int t, auto tag) {
            constexpr bool slow = decltype(tag)::slow;
            RL inA{__shfl_up_sync(FULL, oA.r, 1), __shfl_up_sync(FULL, oA.l, 1)};
            RL inB{__shfl_up_sync(FULL, oB.r, 1), __shfl_up_sync(FULL, oB.l, 1)};
            if (lane == 0) {
                const uint4 qv = vin_s[t];
                inA.r = __uint_as_float(qv.x); inA.l = __uint_as_float(qv.y); inB.r = __uint_as_float(qv.z); inB.l = __uint_as_float(qv.w);
            }
            XRow<D> xa, xb;
            load_x2<D>(xs_lane, 2 * t, xa, xb);
            const int i0 = RP * (c * CH + t - lane);
            if (!slow || (unsigned)i0 < (unsigned)n) {
                float rd = dprev.r, rl = inA.r, ld = dprev.l, ll = inA.l;
#pragma unroll
                for (int w = 0; w < W; ++w) dtw_cell<D, SUB>(xa, z[w], rd, ld, ru[w], lu[w], rl, ll);
                oA.r = rl; oA.l = ll;
                if (SUB && last_strip) track(i0);
            }
            if (!slow || (unsigned)(i0 + 1) < (unsigned)n) {
                float rd = inA.r, rl = inB.r, ld = inA.l, ll = inB.l;
#pragma unroll
                for (int w = 0; w < W; ++w) dtw_cell<D, SUB>(xb, z[w], rd, ld, ru[w], lu[w], rl, ll);
                oB.r = rl; oB.l = ll;
                if (SUB && last_strip) track(i0 + 1);
            }
            dprev = inB;
            if (lane == 31) vout_s[t] = make_uint4(__float_as_uint(oA.r), __float_as_uint(oA.l), __float_as_uint(oB.r), __float_as_uint(oB.l));
        };

        stage_x_async<D>(xs0, p.X, pm.x_off, n, 0, lane);
        const int vlane = (lane < CH) ? lane : 0;
        // column 0 of the border: r_i0 = +inf; Sub-DTW: r_i0 = 0, and a path that enters row i from it starts at row i
        // (the entry of row r is the diagonal predecessor of row r + 1, so it carries r + 1)
        auto border = [&](const int r) {
            return SUB ? make_uint4(0u, __float_as_uint((float)(r + 1)), 0u, __float_as_uint((float)(r + 2))) : make_uint4(F_INF, 0u, F_INF, 0u);
        };
        uint4 vreg = border(2 * vlane);
        bool vbad = false;
        // (r, len) of rows rb, rb + 1 (rb = c CROWS + 2 vlane) from the left strip: column or ring; rows >= n are never used
        auto load_in = [&](const int c) {
            const int rb = c * CROWS + 2 * vlane;
            if (in_ring) {
                const unsigned e = in_q + (unsigned)(c * CH + vlane);
                const unsigned long long* q = ring_of((mypos + FW - 1) % FW) + (size_t)(e & (DTW_RING_ENTRIES - 1)) * 4;
                unsigned long long a0, a1, a2, a3;
                ld_relaxed_v2u64(q, a0, a1);
                ld_relaxed_v2u64(q + 2, a2, a3);
                const unsigned tag = e / DTW_RING_ENTRIES + 1u;
                vreg = make_uint4((unsigned)a0, (unsigned)a1, (unsigned)a2, (unsigned)a3);
                vbad = (rb < n && ((unsigned)(a0 >> 32) != tag || (unsigned)(a1 >> 32) != tag)) ||
                       (rb + 1 < n && ((unsigned)(a2 >> 32) != tag || (unsigned)(a3 >> 32) != tag));
            } else {
                vreg = ld_relaxed_u4(VSprev + 2 * rb);
                vbad = (rb < n && (vreg.x == SENTINEL || vreg.y == SENTINEL)) || (rb + 1 < n && (vreg.z == SENTINEL || vreg.w == SENTINEL));
            }
        };
        if (J > 0) load_in(0);
        unsigned cons_seen = 0;

        for (int c = 0; c < C; ++c) {
            const int rbase = c * CROWS + 2 * vlane;
            if (J > 0) {
                while (__any_sync(FULL, vbad)) {
                    __nanosleep(100);
                    if (vbad) load_in(c);
                }
            }
            cp_async_wait_all();
            if (lane < CH) vin_s[lane] = vreg;
            __syncwarp();
            if (in_ring && lane == 0) st_relaxed_u32(prog_of(mypos), in_q + (unsigned)((c + 1) * CH));   // chunk c taken
            if (out_ring && lane == 0) cons_seen = ld_relaxed_u32(prog_of((mypos + 1) % FW));           // looked at below
            if (c + 1 < C) {
                stage_x_async<D>(xs0 + ((c + 1) & 1) * XWIN * D, p.X, pm.x_off, n, c + 1, lane);
                if (J > 0) load_in(c + 1); else vreg = border(rbase + CROWS);
            }
            xs_lane = xs0 + (c & 1) * XWIN * D + (XPAD - 2 * lane) * D;
            if (interior_chunk(c, n)) {
#pragma unroll 4
                for (int t = 0; t < CH; ++t) step(c, t, FastTag{});
            } else {
#pragma unroll 1
                for (int t = 0; t < CH; ++t) step(c, t, SlowTag{});
            }
            __syncwarp();
            // lane 31 worked on rows c CROWS - SKEW + 2t (+1) at step t
            if (out_ring) {
                // the highest entry of this chunk reuses the slot of the entry RING_ENTRIES below it (of this strip or of the
                // strip before): my consumer must have taken it
                const unsigned need = out_q + (unsigned)((c - DTW_RING_CHUNKS + 1) * CH);
                unsigned seen = __shfl_sync(FULL, cons_seen, 0);
                while ((int)(seen - need) < 0) {
                    __nanosleep(64);
                    if (lane == 0) cons_seen = ld_relaxed_u32(prog_of((mypos + 1) % FW));
                    seen = __shfl_sync(FULL, cons_seen, 0);
                }
                const int q = c * CH - (SKEW / 2) + lane;               // r / 2 for r = c CROWS - SKEW + 2 lane
                if (lane < CH && q >= 0) {
                    const unsigned e = out_q + (unsigned)q;
                    const unsigned long long tag = (unsigned long long)(e / DTW_RING_ENTRIES + 1u) << 32;
                    const uint4 vo = vout_s[lane];
                    unsigned long long* dst = ring_of(mypos) + (size_t)(e & (DTW_RING_ENTRIES - 1)) * 4;
                    st_relaxed_v2u64(dst, tag | vo.x, tag | vo.y);
                    st_relaxed_v2u64(dst + 2, tag | vo.z, tag | vo.w);
                }
            } else if (!out_none) {
                if (lane < CH) st_relaxed_u4(VSme + 2 * (c * CROWS - SKEW + 2 * lane), vout_s[lane]);
            }
        }
        if (in_ring) in_q += (unsigned)(C * CH);
        if (out_ring) out_q += (unsigned)(C * CH);
        // rows >= n were never touched, so ru / lu hold row n of every column: r_{n,m} sits in column m - 1
#pragma unroll
        for (int w = 0; w < W; ++w) {
            if (j0 + w == m - 1) {
                if (SUB) {
                    if (p.out_dtw) p.out_dtw[pm.k] = best;
                    if (p.out_len) p.out_len[pm.k] = (int)best_a;
                    if (p.out_b) p.out_b[pm.k] = best_b;
                } else {
                    if (p.out_dtw) p.out_dtw[pm.k] = ru[w];
                    if (p.out_len) p.out_len[pm.k] = (int)lu[w];
                    if (p.out_score) p.out_score[pm.k] = __fdiv_rn(ru[w], lu[w]);
                }
            }
        }
        __syncwarp();
    }
}

}  // namespace sdtw
