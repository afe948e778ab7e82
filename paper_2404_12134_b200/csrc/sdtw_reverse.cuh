// sdtw_reverse.cuh -- the reverse pass: expected-alignment matrix E of eq. 6
// by recompute + probability flow, fused with the gradient contraction.  Arithmetic: sdtw_kernels.cuh (`cell`).
//
// Decomposition.  A work item is one column strip of one pair (as in the forward kernel) but it is swept by a CTA of
// RW = CH / TR warps: warp b owns BLOCK b (the TR steps b TR .. b TR + TR-1) of every chunk of the strip.  A block is a
// self-contained piece of work: restore its checkpoint, recompute its TR steps keeping every cell's two transition
// weights in shared memory, then run the E recurrence over the same steps backwards.  Only the second half depends on
// the rest of the strip (the E flow that enters the block from below and from the right), so
//   * the recomputes of the RW blocks of a chunk run IN PARALLEL on the CTA's warps, and a warp recomputes its block of
//     the next chunk (speculatively: "the chunk above will be visited too") while the other warps run their flow turns;
//   * the flow state (W accumulators + 3 message registers per lane) is handed from warp to warp through shared
//     memory and an mbarrier per warp ("your turn"): block 3 -> 2 -> 1 -> 0 of chunk c, then block 3 of the next chunk.
// The dependency chain of a pair therefore holds the flow passes only (about a fifth of a chunk's work); in the
// one-warp-per-strip kernel this replaces, the recompute sat on that chain too and a pair's reverse sweep took as long as
// its forward sweep whatever the number of idle SMs.
//
// Exact zero-skip: a chunk whose incoming flows are all +0 leaves every result unchanged and is not
// visited.  Warp 0 is the strip's DECIDER: after its own flow turn it knows the flow state that leaves the chunk,
// looks at the messages of the chunks above (skipping those that carry only +0) and ANNOUNCES the next visited chunk
// to the other warps (or the end of the item).  The first visited chunk of a strip is published to the left
// neighbour as a HINT: a strip's input is +0 in every chunk below (with a larger index than) the first chunk its right
// neighbour visited, so the left strip starts there instead of walking -- and waiting for -- hundreds of zero messages.
//
// Messages between strips are the ones of the kernel this replaces: ES[row] preset to the sentinel pattern, relaxed
// stores by the right strip's lane 0, data-word polling by the left strip; an item ends with a release of its
// progress word FIN | z ("done; every message of my chunks [0, z) is an implicit +0").
#pragma once
#include "sdtw_kernels.cuh"

namespace sdtw {

constexpr int RW = CH / TR;            // warps per CTA of the reverse kernel = blocks per chunk
constexpr int XB = 96;                 // rows of the cycle one block touches: 2 TR rows + the lane skew (62), padded
static_assert(XB >= 2 * TR + SKEW + 2 && XB % 32 == 0, "block window");
constexpr unsigned FIN = 0x80000000u;

struct RevCtl {
    unsigned long long turn[RW];       // mbarriers: "warp b, it is your flow turn"
    unsigned long long ann_bar;        // mbarrier: "announcement i has been made"
    int ann[4];                        // ring of announced visited chunks (-1 = the item has no further visited chunk)
    int item;                          // current work item, or -1: queue empty
};

// floats of dynamic shared memory per warp: weight stash, two block windows of the cycle, vin / ein / eout (TR pairs each)
template <int D> __host__ __device__ constexpr int rev_warp_floats() { return TR * RP * W * 32 * 2 + 2 * XB * D + 3 * 2 * TR; }
// ... plus, per CTA, the flow-state slot (W + 3 values per lane)
template <int D> __host__ __device__ constexpr int rev_smem_bytes() { return (RW * rev_warp_floats<D>() + (W + 3) * 32) * 4; }

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {     // release.cta
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {   // acquire.cta
    unsigned ok = 0;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!ok);
}

// rows [wb, wb + XB) of the scaled cycle -> xs[XB][D]; rows outside [0, n) read as 0
template <int D>
__device__ __forceinline__ void stage_block_async(float* xs, const float* __restrict__ Xs, long long x_off, int n, int wb, int lane) {
    constexpr int VE = (D % 4 == 0) ? 4 : (D % 2 == 0) ? 2 : 1;
    constexpr int PER_LANE = XB * D / VE / 32;
    static_assert(XB * D % (VE * 32) == 0, "whole copies per lane");
#pragma unroll
    for (int q = 0; q < PER_LANE; ++q) {
        const int f = (lane + 32 * q) * VE;
        const int r = wb + f / D;
        const bool ok = (unsigned)r < (unsigned)n;
        const float* src = ok ? Xs + (x_off + wb) * D + f : Xs;
        cp_async<VE * 4>(xs + f, src, ok);
    }
}

template <int D>
__global__ void __launch_bounds__(RW * 32) reverse_kernel(const Params p) {
    extern __shared__ __align__(16) float smem[];
    __shared__ RevCtl ctl;
    const int lane = threadIdx.x & 31, b = threadIdx.x >> 5;               // warp b owns block b of every chunk
    float* wbase = smem + b * rev_warp_floats<D>();
    float2* stash = reinterpret_cast<float2*>(wbase) + lane;                // [TR][RP][W][32] (+ lane)
    float* xsbuf = wbase + TR * RP * W * 32 * 2;                            // [2][XB][D]
    float2* vin_s = reinterpret_cast<float2*>(xsbuf + 2 * XB * D);          // [TR] v_in of lane 0
    float2* ein_s = vin_s + TR;                                             // [TR] messages into lane 31
    float2* eout_s = ein_s + TR;                                            // [TR] messages out of lane 0
    float* slot = smem + RW * rev_warp_floats<D>();                         // [W + 3][32] flow state in transit
    const int m = p.m;
    const int t0 = b * TR;                                                  // first step of my block within a chunk

    if (threadIdx.x == 0) {
        for (int w = 0; w < RW; ++w) mbar_init(&ctl.turn[w], 1);
        mbar_init(&ctl.ann_bar, 1);
    }
    __syncthreads();
    unsigned n_turn = 0;       // flow turns this warp has waited for (parity of its mbarrier)
    unsigned n_ann = 0;        // announcements seen (warps 1..) or made (warp 0)

    for (;;) {
        // Work queue in order of READINESS: the first N entries are the right-most strips of the pairs; every other strip is
        // appended by its right neighbour when that one announces its first visited chunk (or its end), which is when
        // the strip's hint exists.  So a CTA never sits on a strip that cannot start yet: with three CTAs per SM there
        // are only 4.4 strips in flight per pair on cfg 4, and a pair's chain needs about 3.5 of them working.
        if (threadIdx.x == 0) {
            const unsigned q = atomicAdd(p.counters + 1, 1u);
            int it = -1;
            if (q < (unsigned)p.N) it = (int)q * p.NS + p.NS - 1;
            else if (q < p.num_items) {
                unsigned v;
                while ((v = ld_relaxed_u32(p.ready_b + (q - p.N))) == 0u) __nanosleep(64);
                it = (int)v - 1;
            }
            ctl.item = it;
        }
        __syncthreads();
        const int item = ctl.item;
        if (item < 0) break;
        const int ps = item / p.NS, J = item - ps * p.NS;
        const PairMeta pm = p.pm[ps];
        const int n = pm.n, C = pm.C;
        const int j0 = (J * 32 + lane) * W;
        const bool has_right = (J < p.NS - 1);
        const int band = p.band;
        const bool dense = p.dense_reverse != 0;
        int cf, cl;                                           // chunks of this strip with rows inside the band
        band_chunks(J, band, C, cf, cl);
        const int bfirst = cf * RW;
        const float* VSprev = p.VS + pm.vs_off + (long long)(J - 1) * pm.vs_stride + VS_PAD;
        float* ESme = p.ES + pm.vs_off + (long long)J * pm.vs_stride + VS_PAD;   // indexed by row
        const float* ESnext = ESme + pm.vs_stride;
        const float* CKme = p.CK + pm.ck_off + (long long)J * pm.ck_stride;

        float z[W][D], g[W][D], A[W], h[W];
#pragma unroll
        for (int w = 0; w < W; ++w) {
            const int j = j0 + w;
#pragma unroll
            for (int c = 0; c < D; ++c) { z[w][c] = (j < m) ? __ldg(p.Zs + (long long)j * D + c) : 0.f; g[w][c] = 0.f; }
            A[w] = 0.f; h[w] = 0.f;
        }
        float vp0 = 0.f, vp1 = 0.f;
        float msg0_prev = 0.f, msg1_prev = 0.f, cdf_prev = 0.f;

        // ---- loads of one block (chunk c): cycle rows (cp.async), checkpoint, v_in of lane 0, messages into lane 31
        float4 ph[W / 4]; float2 pv = make_float2(0.f, 0.f);
        float2 vreg = make_float2(0.f, 0.f), ereg = make_float2(0.f, 0.f);
        int loaded = -1;                                       // chunk whose loads are in flight / in registers
        auto msg_row = [&](const int c) { return c * CROWS - SKEW + 2 * (t0 + lane); };   // lane u < TR: pair of step t0 + u
        auto issue_loads = [&](const int c) {
            if (loaded >= 0) cp_async_wait_all();              // an unused speculative load may still be landing in this buffer
            const int bidx = c * RW + b;
            stage_block_async<D>(xsbuf + (c & 1) * XB * D, p.Xs, pm.x_off, n, c * CROWS + 2 * t0 - 64, lane);
            if (bidx > bfirst) {                               // block bfirst starts from the zero state, not a checkpoint
                const float* ck = CKme + (long long)bidx * CK_FLOATS;
#pragma unroll
                for (int gq = 0; gq < W / 4; ++gq) ph[gq] = __ldcs(reinterpret_cast<const float4*>(ck) + gq * 32 + lane);
                pv = __ldcs(reinterpret_cast<const float2*>(ck + W * 32) + lane);
            }
            if (lane < TR) {
                const int rbase = c * CROWS + 2 * (t0 + lane);
                vreg = (J > 0) ? __ldcs(reinterpret_cast<const float2*>(VSprev + rbase)) : make_float2(rbase == 0 ? BIG : 0.f, 0.f);
                const int r = msg_row(c);
                ereg = (has_right && r >= 0) ? ld_relaxed_f2(ESnext + r) : make_float2(0.f, 0.f);
            }
            loaded = c;
        };

        // ---- recompute of my block of chunk c: weights -> stash
        auto rec_row = [&](const int i, const XRow<D>& x, float& v, const int slot_) {
#pragma unroll
            for (int w = 0; w < W; ++w) {
                float tl, acc, wu, wl;
                sqdist2<D>(x, z[w], tl, acc);
                if (band >= 0) {                              // band edges, as in the forward kernel
                    if (j0 + w - i == band) h[w] = BIG;
                    if (i - (j0 + w) == band) v = BIG;
                }
                cell<true, (D > 1)>(tl, acc, h[w], v, wu, wl);
                stash[(slot_ * W + w) * 32] = make_float2(wu, wl);
            }
        };
        auto block_fast = [&](const int c) {                   // every cell of the block lies inside the matrix, off the band edges
            const int lo = c * CROWS + 2 * t0 - SKEW, hi = c * CROWS + 2 * (t0 + TR - 1) + 1;
            return lo >= 0 && hi < n && band_clear(c, J, band);
        };
        auto recompute = [&](const int c, float2& ein_out) {
            const int bidx = c * RW + b;
            cp_async_wait_all();
            __syncwarp();                                      // the flow of the chunk before last has finished reading vin_s / xs
            if (lane < TR) vin_s[lane] = vreg;
            ein_out = ereg;
            if (bidx == bfirst) {                              // the forward sweep started here from the zero state
#pragma unroll
                for (int w = 0; w < W; ++w) h[w] = (bidx == 0 && j0 + w == 0) ? BIG : 0.f;
                vp0 = vp1 = 0.f;
            } else {
#pragma unroll
                for (int gq = 0; gq < W / 4; ++gq) { h[4 * gq] = ph[gq].x; h[4 * gq + 1] = ph[gq].y; h[4 * gq + 2] = ph[gq].z; h[4 * gq + 3] = ph[gq].w; }
                vp0 = pv.x; vp1 = pv.y;
            }
            __syncwarp();
            const float* xs_lane = xsbuf + (c & 1) * XB * D + (64 - 2 * lane) * D;   // rows of step t0 + u: xs_lane[2u], [2u + 1]
            if (block_fast(c)) {
#pragma unroll
                for (int u = 0; u < TR; ++u) {
                    float va = __shfl_up_sync(FULL, vp0, 1), vb = __shfl_up_sync(FULL, vp1, 1);
                    if (lane == 0) { const float2 qv = vin_s[u]; va = qv.x; vb = qv.y; }
                    XRow<D> xa, xb;
                    load_x2<D>(xs_lane, 2 * u, xa, xb);
#pragma unroll
                    for (int w = 0; w < W; ++w) {
                        float tl, acc, wu, wl;
                        sqdist2<D>(xa, z[w], tl, acc);
                        cell<true, (D > 1)>(tl, acc, h[w], va, wu, wl);
                        stash[((u * RP + 0) * W + w) * 32] = make_float2(wu, wl);
                        sqdist2<D>(xb, z[w], tl, acc);
                        cell<true, (D > 1)>(tl, acc, h[w], vb, wu, wl);
                        stash[((u * RP + 1) * W + w) * 32] = make_float2(wu, wl);
                    }
                    vp0 = va; vp1 = vb;
                }
            } else {
#pragma unroll 1
                for (int u = 0; u < TR; ++u) {
                    float va = __shfl_up_sync(FULL, vp0, 1), vb = __shfl_up_sync(FULL, vp1, 1);
                    if (lane == 0) { const float2 qv = vin_s[u]; va = qv.x; vb = qv.y; }
                    XRow<D> xa, xb;
                    load_x2<D>(xs_lane, 2 * u, xa, xb);
                    const int i0 = RP * (c * CH + t0 + u - lane);
                    if ((unsigned)i0 < (unsigned)n) { rec_row(i0, xa, va, u * RP + 0); vp0 = va; }
                    if ((unsigned)(i0 + 1) < (unsigned)n) { rec_row(i0 + 1, xb, vb, u * RP + 1); vp1 = vb; }
                }
            }
            loaded = -1;
        };

        // ---- E recurrence of one row, right to left (probability flow; mass conserving)
        auto e_row = [&](const XRow<D>& x, const float e_in, const int slot_, float& cl_, float& cd) {
            float E = A[W - 1] + e_in;
            float cd_right = 0.f;
#pragma unroll
            for (int w = W - 1; w >= 0; --w) {
                const float2 wt = stash[(slot_ * W + w) * 32];
#pragma unroll
                for (int ch = 0; ch < D; ++ch) g[w][ch] = fmaf(E, z[w][ch] - x.c[ch], g[w][ch]);
                const float Anew = fmaf(E, wt.x, cd_right);       // into (i-1, j): from (i, j) and, diagonally, (i, j+1)
                cd_right = fmaf(-E, wt.y, fmaf(-E, wt.x, E));     // diagonal share of this cell
                if (w > 0) E = fmaf(E, wt.y, A[w - 1]); else cl_ = E * wt.y;
                A[w] = Anew;
            }
            cd = cd_right;
        };
        auto flow = [&](const int c) {                         // my block of chunk c, steps t0 + TR-1 .. t0
            const float* xs_lane = xsbuf + (c & 1) * XB * D + (64 - 2 * lane) * D;
            if (block_fast(c)) {                               // no bounds tests: the loads of a step can be hoisted freely
#pragma unroll
                for (int u = TR - 1; u >= 0; --u) {
                    float in0 = __shfl_down_sync(FULL, msg0_prev, 1), in1 = __shfl_down_sync(FULL, msg1_prev, 1);
                    if (lane == 31) { const float2 qe = ein_s[u]; in0 = qe.x; in1 = qe.y; }
                    XRow<D> xa, xb;
                    load_x2<D>(xs_lane, 2 * u, xa, xb);
                    float cl1, cd1, cl0, cd0;
                    e_row(xb, in1, u * RP + 1, cl1, cd1);
                    msg1_prev = cl1 + cdf_prev;                // into the left neighbour's cell (i0+1, j0-1)
                    e_row(xa, in0, u * RP + 0, cl0, cd0);
                    msg0_prev = cl0 + cd1;                     // into (i0, j0-1)
                    cdf_prev = cd0;
                    if (lane == 0) eout_s[u] = make_float2(msg0_prev, msg1_prev);
                }
            } else {
#pragma unroll 1
                for (int u = TR - 1; u >= 0; --u) {
                    float in0 = __shfl_down_sync(FULL, msg0_prev, 1), in1 = __shfl_down_sync(FULL, msg1_prev, 1);
                    if (lane == 31) { const float2 qe = ein_s[u]; in0 = qe.x; in1 = qe.y; }
                    XRow<D> xa, xb;
                    load_x2<D>(xs_lane, 2 * u, xa, xb);
                    const int i0 = RP * (c * CH + t0 + u - lane);
                    float cd_mid = cdf_prev;                   // row i0+1 missing (i0 + 1 == n): its diagonal share is 0
                    if ((unsigned)(i0 + 1) < (unsigned)n) {
                        float cl1, cd1;
                        e_row(xb, in1, u * RP + 1, cl1, cd1);
                        msg1_prev = cl1 + cdf_prev;
                        cd_mid = cd1;
                    }
                    if ((unsigned)i0 < (unsigned)n) {
                        float cl0, cd0;
                        e_row(xa, in0, u * RP + 0, cl0, cd0);
                        msg0_prev = cl0 + cd_mid;
                        cdf_prev = cd0;
                    }
                    if (lane == 0) eout_s[u] = make_float2(msg0_prev, msg1_prev);
                }
            }
        };
        auto put_state = [&]() {
#pragma unroll
            for (int w = 0; w < W; ++w) slot[w * 32 + lane] = A[w];
            slot[W * 32 + lane] = msg0_prev; slot[(W + 1) * 32 + lane] = msg1_prev; slot[(W + 2) * 32 + lane] = cdf_prev;
        };
        auto get_state = [&]() {
#pragma unroll
            for (int w = 0; w < W; ++w) A[w] = slot[w * 32 + lane];
            msg0_prev = slot[W * 32 + lane]; msg1_prev = slot[(W + 1) * 32 + lane]; cdf_prev = slot[(W + 2) * 32 + lane];
        };

        // ---- the right strip's progress word and messages
        unsigned finw = 0;                                     // the right strip's progress word as last seen
        auto poll_fin = [&]() {
            if (has_right && !(finw & FIN)) {
                unsigned f = 0;
                if (lane == 0) f = ld_acquire(p.prog_b + item + 1);
                finw = __shfl_sync(FULL, f, 0);
                __syncwarp();                                  // the other lanes reload ES only after lane 0's acquire
            }
        };
        // wait until the message pair `e` of row `r` (lanes with `mine`) is published, or known to be an implicit +0.
        // The data words are polled back to back (detection delay = one L2 round trip); the right strip's progress word
        // is looked at only now and then.
        auto resolve = [&](float2& e, const int r, const bool mine) {
            bool bad = mine && (is_sentinel(e.x) || is_sentinel(e.y));
            unsigned it = 0;
            while (__any_sync(FULL, bad)) {
                if (bad) {
                    e = ld_relaxed_f2(ESnext + r);
                    bad = is_sentinel(e.x) || is_sentinel(e.y);
                }
                if (!__any_sync(FULL, bad)) break;
                if ((++it & 3u) == 0u || (finw & FIN)) {
                    poll_fin();
                    // the right strip is done and this row lies in a chunk it never visited: never written
                    if (bad && (finw & FIN) && r / CROWS < (int)(finw & ~FIN)) { e = make_float2(0.f, 0.f); bad = false; }
                }
            }
        };

        // ---- decisions (warp 0): next visited chunk at or above `c`, given the flow state in this warp's registers
        unsigned long long visited = 0;
        bool hinted = false;
        int c_ann = -1;                                        // the last announcement (warp 0 keeps its own copy)
        auto announce = [&](const int c) {
            if (lane == 0) {
                ctl.ann[n_ann & 3] = c;
                mbar_arrive(&ctl.ann_bar);
                if (!hinted && J > 0) {
                    // first visited chunk of this strip: the left strip's input is +0 in every chunk with a larger index;
                    // the left strip can start now (or, if this strip ends without a visit, has nothing to do): queue it
                    if (c >= 0) st_relaxed_u32(p.hint_b + item, (unsigned)c + 1u);
                    st_relaxed_u32(p.ready_b + atomicAdd(p.counters + 2, 1u), (unsigned)item);   // item - 1, stored + 1
                }
            }
            hinted = true;
            c_ann = c;
            ++n_ann;
        };
        int z_fin = cl + 1;                                    // chunks [0, z_fin) of this item carry implicit +0 messages
        auto decide = [&](int c) -> int {
            for (; c >= cf; --c) {
                unsigned lbits = __float_as_uint(msg0_prev) | __float_as_uint(msg1_prev) | __float_as_uint(cdf_prev);
#pragma unroll
                for (int w = 0; w < W; ++w) lbits |= __float_as_uint(A[w]);
                if (dense || __any_sync(FULL, lbits != 0u)) return c;       // flow already inside this strip
                if (!has_right) break;                         // nothing inside, nothing can arrive: the item is over
                // all 32 message pairs of chunk c (lane t: the pair of lane 31's step t) and a peek at the right strip's end
                const int r = c * CROWS - SKEW + 2 * lane;
                float2 e = (r >= 0) ? ld_relaxed_f2(ESnext + r) : make_float2(0.f, 0.f);
                unsigned pk = 0;
                if (lane == 0 && !(finw & FIN)) pk = ld_relaxed_u32(p.prog_b + item + 1);
                if (__shfl_sync(FULL, pk, 0) & FIN) poll_fin();              // make it official (acquire)
                if ((finw & FIN) && c < (int)(finw & ~FIN)) break;          // the rest are implicit zeros: the item is over
                resolve(e, r, r >= 0);
                if ((finw & FIN) && c < (int)(finw & ~FIN)) break;
                const unsigned bits = __float_as_uint(e.x) | __float_as_uint(e.y);
                if (__any_sync(FULL, bits != 0u)) return c;
                if (J > 0) st_relaxed_f2(ESme + c * CROWS + 2 * lane, make_float2(0.f, 0.f));   // exact skip: forward the zeros
            }
            z_fin = max(c + 1, cf);
            return -1;
        };

        // ---- item start: warp 0 finds where its decisions start
        int c_try = cl;                                        // warp 0: the next decision starts at this chunk
        if (b == 0) {
            if (J == p.NS - 1) {
#pragma unroll
                for (int w = 0; w < W; ++w) A[w] = (j0 + w == m - 1) ? 1.f : 0.f;    // E[n+1][m+1] = 1 flows into cell (n, m)
            } else if (!dense) {
                // The input of this strip is +0 in every chunk with a larger index than the first chunk the right strip
                // visits: wait for that hint (or for the right strip to finish without having visited anything).
                unsigned hv = 0, spins = 0;
                for (;;) {
                    if (lane == 0) hv = ld_relaxed_u32(p.hint_b + item + 1);
                    hv = __shfl_sync(FULL, hv, 0);
                    if (hv) break;
                    if ((++spins & 7u) == 0u) {
                        poll_fin();
                        if (finw & FIN) {                      // finished: a hint stored before the release is visible now
                            if (lane == 0) hv = ld_relaxed_u32(p.hint_b + item + 1);
                            hv = __shfl_sync(FULL, hv, 0);
                            break;
                        }
                    }
                    __nanosleep(32);
                }
                c_try = hv ? min(cl, (int)hv - 1) : -2;        // -2: the right strip never carried any flow, nor will this one
            }
        }
        auto wait_ann = [&]() {
            mbar_wait(&ctl.ann_bar, n_ann & 1);
            const int c = ctl.ann[n_ann & 3];
            ++n_ann;
            return c;
        };

        // ---- the chunk loop: announcement -> (recompute) -> flow turn -> hand over; a warp recomputes its block of the
        // chunk above speculatively while the other warps take their flow turns.  `recompute` and `flow` are each
        // instantiated ONCE (the kernel is instruction-cache bound otherwise).
        bool spec = false;                                     // warps 1..: c_rec is a guess, not an announcement
        int c_rec = -1;
        float2 ein_cur = make_float2(0.f, 0.f);
        for (;;) {
            int c;
            if (b == 0) {
                if (c_try == -2) { c = -1; z_fin = cl + 1; } else c = decide(c_try);
                if (c >= 0) { put_state(); __syncwarp(); }
                announce(c);
                if (c < 0) break;
                if (lane == 0) mbar_arrive(&ctl.turn[RW - 1]);
            } else if (spec) {
                c = c_rec;
            } else {
                c = wait_ann();
                if (c < 0) break;
            }
            for (;;) {                                         // at most two passes: a wrong guess is recomputed
                if (loaded != c) issue_loads(c);
                recompute(c, ein_cur);
                if (c - 1 >= cf) issue_loads(c - 1);            // guess: the chunk above is visited as well
                if (!spec) break;
                spec = false;
                const int ca = wait_ann();
                if (ca == c) break;
                c = ca;
                if (c < 0) break;
            }
            if (c < 0) break;
            ++visited;
            const int cs = c - 1;
            // my flow turn
            mbar_wait(&ctl.turn[b], n_turn & 1);
            ++n_turn;
            get_state();
            resolve(ein_cur, msg_row(c), has_right && lane < TR && msg_row(c) >= 0);
            if (lane < TR) ein_s[lane] = ein_cur;
            __syncwarp();
            flow(c);
            __syncwarp();
            // lane 0 worked on rows 64 c + 2 t (+1) at step t
            if (J > 0 && lane < TR) st_relaxed_f2(ESme + c * CROWS + 2 * (t0 + lane), eout_s[lane]);
            if (b > 0) {
                put_state();
                __syncwarp();
                if (lane == 0) mbar_arrive(&ctl.turn[b - 1]);
                spec = (cs >= cf);
                c_rec = cs;
            } else {
                c_try = cs;
            }
        }
        if (loaded >= 0) { cp_async_wait_all(); loaded = -1; }   // a speculative load nobody used

        // ---- end of the item: sum the warps' partial contractions (fixed order), publish FIN, write Gk
        float* gsum = wbase;                                   // my stash is free now: [W * D][32]
#pragma unroll
        for (int w = 0; w < W; ++w)
#pragma unroll
            for (int ch = 0; ch < D; ++ch) gsum[(w * D + ch) * 32 + lane] = g[w][ch];
        __syncthreads();
        if (b == 0) {
            if (lane == 0) {
                st_release(p.prog_b + item, FIN | (unsigned)z_fin);
                if (p.stats) { atomicAdd(p.stats + 0, (unsigned long long)C); atomicAdd(p.stats + 1, (unsigned long long)C - visited); }
            }
#pragma unroll
            for (int w = 0; w < W; ++w) {
                const int j = j0 + w;
                if (j < m) {
#pragma unroll
                    for (int ch = 0; ch < D; ++ch) {
                        float s = 0.f;
#pragma unroll
                        for (int bb = RW - 1; bb >= 0; --bb) s += smem[bb * rev_warp_floats<D>() + (w * D + ch) * 32 + lane];
                        p.Gk[((long long)ps * m + j) * D + ch] = s * p.gscale;   // eq. 6 partial of this pair, natural units
                    }
                }
            }
        }
        __syncthreads();                                       // the stashes are read above; the next item overwrites them
    }
}

}  // namespace sdtw
