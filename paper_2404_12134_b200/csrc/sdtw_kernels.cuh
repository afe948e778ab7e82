// sdtw_kernels.cuh -- sm_100a kernels of the Soft-DTW value / gradient path (DESIGN.md sections 5-6).
//
// Formulation (all in "scaled units": inputs are multiplied by sqrt(kappa), kappa = 1/(gamma ln 2), so that
// min^gamma of eq. 3 becomes -log2 sum 2^(-a) and no multiply by gamma appears per cell):
//
//   difference form of eq. 5:  h[i][j] = r[i][j] - r[i][j-1],  v[i][j] = r[i][j] - r[i-1][j]
//     s      = softmin(0, h_in, v_in),  h_in = h[i-1][j], v_in = v[i][j-1]   (relative to the diagonal predecessor)
//     h[i][j] = D + s - v_in,  v[i][j] = D + s - h_in
//   the three transition weights of the reverse recurrence (eq. 6's E) are the softmax terms
//     (w_diag, w_up, w_left) = (1, 2^-h_in, 2^-v_in) / (1 + 2^-h_in + 2^-v_in)
//   and E is pushed backwards as a probability flow:  E[pred] += E[cell] * w_pred  (mass conserving in fp32).
//
// Work decomposition: a WORK ITEM is one column strip (32 lanes x W columns) of one pair, swept over all rows by ONE
// warp.  At step s lane l works on the RP = 2 rows 2(s - l), 2(s - l) + 1 of its W columns: a skewed anti-diagonal
// wavefront whose 2 x W register tile gives every thread two independent dependency chains (the cells (A, w+1) and
// (A+1, w) do not depend on each other), which is what keeps the MUFU pipe fed.  Neighbouring lanes exchange two values
// per step by warp shuffle; neighbouring strips exchange the strip-boundary column through global memory:
//   forward  VS[row]: written by lane 31 of the left strip, read by lane 0 of the right strip.  No flag: the buffer is
//            preset to a sentinel bit pattern no arithmetic result can have and the consumer polls the DATA words with
//            relaxed gpu-scope loads, one 64-row chunk ahead of use, so the wait is normally hidden;
//   reverse  ES[row]: E messages from the right strip to the left one, same protocol (sentinel preset, relaxed data-word
//            polling one chunk ahead); only the END of an item is published with a release (its progress word).
// Every TR steps the forward kernel checkpoints the warp state (h[W] + the two values in flight) to HBM; the reverse
// kernels restore a checkpoint, recompute TR steps keeping the transition weights in shared memory, then run the E
// recurrence over those TR steps backwards, accumulating the gradient contraction of eq. 6 in registers.  This file
// holds the throughput-regime reverse kernel (backward_kernel: one warp per strip); sdtw_reverse.cuh holds the
// latency-regime one (reverse_kernel: a CTA of four warps per strip).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sdtw {

#ifndef SDTW_W
#define SDTW_W 4
#endif
#ifndef SDTW_TR
#define SDTW_TR 8
#endif
#ifndef SDTW_WARPS
#define SDTW_WARPS 4
#endif
#ifndef SDTW_CH
#define SDTW_CH 32
#endif

constexpr int W = SDTW_W;       // columns per thread
constexpr int RP = 2;           // rows per lane per step
constexpr int SW = 32 * W;      // columns per strip (work item)
constexpr int CH = SDTW_CH;     // steps per chunk (granularity of the strip-boundary exchange), <= 32
constexpr int CROWS = CH * RP;  // rows a lane sweeps per chunk
constexpr int SKEW = 31 * RP;   // lane 31 is this many rows behind lane 0
constexpr int XPAD = 64;        // >= SKEW, keeps the staged window aligned
constexpr int XWIN = XPAD + CROWS;  // rows of the cycle staged per chunk: [c*CROWS - XPAD, c*CROWS + CROWS)
constexpr int LAGC = (SKEW + CROWS - 1) / CROWS;  // chunks of the neighbouring strip one chunk reaches back into
constexpr int TR = SDTW_TR;     // steps between checkpoints (= steps recomputed per reverse block)
constexpr int WARPS = SDTW_WARPS;  // warps per CTA (each warp is an independent agent)
constexpr int CK_FLOATS = 32 * (W + RP);  // floats per checkpoint record
constexpr int VS_PAD = 64;      // floats of front padding of every VS / ES strip (rows -62 .. -1 are addressed)
constexpr float BIG = 1.0e30f;  // stands for the +inf border of eq. 5
constexpr unsigned FULL = 0xffffffffu;
constexpr unsigned SENTINEL = 0xffffffffu;  // a NaN pattern no arithmetic instruction returns (results are 0x7fffffff)

static_assert(W % 4 == 0, "checkpoints store h as float4");
static_assert(CH % TR == 0 && CH <= 32, "a chunk holds a whole number of checkpoint blocks; one lane per step");
static_assert(VS_PAD >= SKEW && XPAD >= SKEW && (XWIN * 1) % 32 == 0, "padding covers the lane skew");

constexpr int RING_CHUNKS = 16;                    // chunks a producer may run ahead of its consumer inside a unit
constexpr int RING_ENTRIES = RING_CHUNKS * CH;     // ring entries (one per pair of rows), a power of two
static_assert((RING_ENTRIES & (RING_ENTRIES - 1)) == 0, "ring size is a power of two");

struct PairMeta {   // one per pair, in schedule order (longest first)
    long long x_off;      // first row of this cycle in X_concat
    long long vs_off;     // float offset of strip 0's boundary column in VS / ES; strip stride = vs_stride
    long long ck_off;     // float offset of strip 0's checkpoints; strip stride = ck_stride
    long long ck_stride;
    int vs_stride;
    int n;                // rows of this cycle
    int k;                // caller's pair index
    int C;                // chunks = ceil((ceil(n / RP) + 31) / CH)
};

struct Params {
    const float* Zs;      // sqrt(kappa) * Z
    const float* Xs;      // sqrt(kappa) * X_concat
    const PairMeta* pm;
    unsigned* counters;   // [0] forward work queue, [1] reverse work queue (head), [2] tail of ready_b
    unsigned* prog_b;     // [N * NS] progress word of each reverse item: FIN | z when it is done
    unsigned* hint_b;     // [N * NS] 1 + the first chunk the reverse item visited (0: none yet)
    unsigned* ready_b;    // [N * NS] reverse_kernel's work queue behind the first N entries: 1 + item, in order of readiness
    float* VS;            // strip-boundary v columns, indexed by row
    float* ES;            // strip-boundary E messages, indexed by row
    float* CK;            // checkpoints
    double* VP;           // [N * NS] per-item partial of the value (staircase sum), scaled units
    float* Gk;            // [N][m][D] per-pair gradient partials
    int m, N, NS;
    unsigned num_items;
    unsigned long long* stats;  // [0] reverse chunks visited, [1] reverse chunks skipped (instrumentation; may be null)
    int dense_reverse;    // 1: never skip a reverse chunk (for measurement / validation of the exact skip)
    int unit_strips;      // forward schedule: adjacent strips of one pair per unit (1 .. warps per CTA)
    int tail_from;        // strips >= tail_from (a multiple of unit_strips, <= NS) are handed out in units of tail_unit
    int tail_unit;        //   strips (>= 1): the last units in the queue are small, which shortens the drain
    int band;             // Sakoe-Chiba band (Table 1): cell (i, j) admissible iff |i - j| <= band; < 0: none
    // forward-only sweeps (no checkpoints): strip-boundary values travel through small rings inside a unit (null: every
    // boundary has a full column, as in the gradient path); see forward_kernel
    unsigned long long* ring;   // [CTA][warp position][RING_ENTRIES][2]: (value bits | tag << 32) per row
    unsigned* ring_prog;        // [CTA][warp position] entries of the left neighbour's ring this warp has consumed
    const float* wts;     // [N] per-pair weights of eq. 7 in schedule order, or null (all 1)
    float gscale;         // 2 / sqrt(kappa)
};

__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float lg2_approx(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp_approx(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ unsigned ld_acquire(const unsigned* p) {
    unsigned v; asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v;
}
__device__ __forceinline__ void st_release(unsigned* p, unsigned v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// relaxed gpu-scope accesses of the forward strip-boundary column (each 32-bit word is valid or the sentinel)
__device__ __forceinline__ float2 ld_relaxed_f2(const float* p) {
    float2 v; asm volatile("ld.relaxed.gpu.global.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p) : "memory"); return v;
}
__device__ __forceinline__ void st_relaxed_f2(float* p, float2 v) {
    asm volatile("st.relaxed.gpu.global.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ unsigned ld_relaxed_u32(const unsigned* p) {
    unsigned v; asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v;
}
__device__ __forceinline__ void st_relaxed_u32(unsigned* p, unsigned v) {
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void ld_relaxed_v2u64(const unsigned long long* p, unsigned long long& a, unsigned long long& b) {
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
}
__device__ __forceinline__ void st_relaxed_v2u64(unsigned long long* p, unsigned long long a, unsigned long long b) {
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(a), "l"(b) : "memory");
}
__device__ __forceinline__ bool is_sentinel(float x) { return __float_as_uint(x) == SENTINEL; }

template <int BYTES>
__device__ __forceinline__ void cp_async(float* smem_dst, const float* gsrc, bool ok) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int sz = ok ? BYTES : 0;                           // src-size 0: the destination is zero-filled
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2, %3;" ::"r"(s), "l"(gsrc), "n"(BYTES), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// shared memory per warp (floats)
template <int D> __host__ __device__ constexpr int fwd_smem_floats() { return 2 * XWIN * D + 4 * 32; }
template <int D> __host__ __device__ constexpr int bwd_smem_floats() { return TR * RP * W * 32 * 2 + XWIN * D + 6 * 32; }

template <int D> struct XRow { float c[D]; };

// rows e and e + 1 (e even) of a staged window
template <int D>
__device__ __forceinline__ void load_x2(const float* xs, int e, XRow<D>& a, XRow<D>& b) {
    if constexpr (D == 1) {
        const float2 t = *reinterpret_cast<const float2*>(xs + e);
        a.c[0] = t.x; b.c[0] = t.y;
    } else if constexpr (D == 2) {
        const float4 t = *reinterpret_cast<const float4*>(xs + e * 2);
        a.c[0] = t.x; a.c[1] = t.y; b.c[0] = t.z; b.c[1] = t.w;
    } else if constexpr (D == 4) {
        const float4 t = *reinterpret_cast<const float4*>(xs + e * 4);
        const float4 u = *reinterpret_cast<const float4*>(xs + e * 4 + 4);
        a.c[0] = t.x; a.c[1] = t.y; a.c[2] = t.z; a.c[3] = t.w;
        b.c[0] = u.x; b.c[1] = u.y; b.c[2] = u.z; b.c[3] = u.w;
    } else {
#pragma unroll
        for (int c = 0; c < D; ++c) { a.c[c] = xs[e * D + c]; b.c[c] = xs[(e + 1) * D + c]; }
    }
}

// asynchronously stage rows [c*CROWS - XPAD, c*CROWS + CROWS) of the scaled cycle into xs[XWIN][D]; rows outside
// [0, n) read as 0.  Completed by cp_async_wait_all() + __syncwarp().
template <int D>
__device__ __forceinline__ void stage_x_async(float* xs, const float* __restrict__ Xs, long long x_off, int n, int c, int lane) {
    constexpr int VE = (D % 4 == 0) ? 4 : (D % 2 == 0) ? 2 : 1;       // floats per copy (a copy never straddles a row)
    constexpr int PER_LANE = XWIN * D / VE / 32;
    static_assert(XWIN * D % (VE * 32) == 0, "whole copies per lane");
    const int wb = c * CROWS - XPAD;
#pragma unroll
    for (int q = 0; q < PER_LANE; ++q) {
        const int f = (lane + 32 * q) * VE;                           // float index in the window
        const int r = wb + f / D;
        const bool ok = (unsigned)r < (unsigned)n;
        const float* src = ok ? Xs + (x_off + wb) * D + f : Xs;
        cp_async<VE * 4>(xs + f, src, ok);
    }
}

// ------------------------------------------------------------------------------------------------------------------
// one cell of the difference-form recurrence.  v is v_in on entry and v_out on return; h is h_in / h_out.
// The cell cost is D = t_last^2 + acc, so that the last square fuses with the subtraction of the log (one FFMA).
// With a = mn - h_in, b = mn - v_in (mn = min(0, h_in, v_in); one of 0, a, b is exactly 0) the three soft-min terms are
// 2^mn (diagonal), 2^a ("up"), 2^b ("left"); sorted, they are 1, e1 = 2^-|min(h,v)| and e2 = 2^min(a,b).
// STASH: also emit the weights (w_up, w_left) of this cell's "up" and "left" predecessors.
__device__ __forceinline__ float min3(float a, float b, float c) {
    float r; asm("min.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r;
}
// 2^x for x <= 0 on the FMA pipe (no MUFU): x = n + f, n = round(x), 2^f by a degree-5 polynomial on [-0.5, 0.5]
// (relative error 2.3e-7 in fp32, the same as ex2.approx), 2^n assembled in the exponent field.  x <= -127 gives +0
// exactly, like ex2.approx.ftz does for the +inf borders (BIG).
__device__ __forceinline__ float ex2_fma(float x) {
    x = fmaxf(x, -127.f);
    const float t = x + 12582912.f;                      // 1.5 * 2^23: n lands in the low mantissa bits
    const float f = x - (t - 12582912.f);
    float q = 0.001327647129073739f;
    q = fmaf(q, f, 0.009675540961325169f);
    q = fmaf(q, f, 0.05550713092088699f);
    q = fmaf(q, f, 0.24022120237350464f);
    q = fmaf(q, f, 0.6931469440460205f);
    q = fmaf(q, f, 1.0000001192092896f);
    return q * __int_as_float((__float_as_int(t) << 23) + 0x3f800000);
}
// Forward kernel only: bit w of the mask set = column w of a thread evaluates its second exponential with ex2_fma
// (mask A: the even row of a step, mask B: the odd row).  The MUFU pipe is the forward kernel's bound and its issue
// slots are 60 % busy, so moving a quarter of the ex2 work to the FMA pipe shortens the sweep.  The reverse kernel is
// latency bound and keeps MUFU for all three (a 12-instruction chain instead of one would lengthen its critical path).
// d >= 3: the cost arithmetic already fills the issue slots, so the polynomial is not used there either.
#ifndef SDTW_POLY_MASK_A
#define SDTW_POLY_MASK_A 2
#endif
#ifndef SDTW_POLY_MASK_B
#define SDTW_POLY_MASK_B 10
#endif
template <bool STASH, bool HASACC>
__device__ __forceinline__ void cell(float t_last, float acc, float& h, float& v, float& wu, float& wl, const bool poly = false) {
    const float hin = h, vin = v;
    const float mn = min3(hin, vin, 0.f);
    const float p = fminf(hin, vin);
    const float a = mn - hin, b = mn - vin;
    const float e1 = ex2_approx(-fabsf(p));     // p >= 0: the min(h,v) term;  p < 0: the diagonal term
    const float e2 = poly ? ex2_fma(fminf(a, b)) : ex2_approx(fminf(a, b));   // the max(h,v) term
    const float S = (1.f + e1) + e2;
    const float l = lg2_approx(S);
    const float c = HASACC ? fmaf(t_last, t_last, acc - l) : fmaf(t_last, t_last, -l);
    h = c + b;
    v = c + a;
    if constexpr (STASH) {
        const float rS = rcp_approx(S);
        const float wp = (p < 0.f) ? rS : e1 * rS;
        const float wq = e2 * rS;
        const bool h_is_p = a >= b;             // h_in <= v_in
        wu = h_is_p ? wp : wq;
        wl = h_is_p ? wq : wp;
    }
}

// cost of one cell as (t_last, acc): D = t_last^2 + acc
template <int D>
__device__ __forceinline__ void sqdist2(const XRow<D>& x, const float (&z)[D], float& t_last, float& acc) {
    acc = 0.f;
#pragma unroll
    for (int c = 0; c + 1 < D; ++c) { const float t = x.c[c] - z[c]; acc = fmaf(t, t, acc); }
    t_last = x.c[D - 1] - z[D - 1];
}

template <int D>
__device__ __forceinline__ float sqdist(const XRow<D>& x, const float (&z)[D]) {
    float t = x.c[0] - z[0];
    float acc = t * t;
#pragma unroll
    for (int c = 1; c < D; ++c) { t = x.c[c] - z[c]; acc = fmaf(t, t, acc); }
    return acc;
}

struct FastTag { static constexpr bool slow = false; static constexpr bool val = false; };
struct SlowTag { static constexpr bool slow = true; static constexpr bool val = true; };
// fast arithmetic (no bounds / band tests) plus the bookkeeping of the value staircase: the chunks a warp's staircase
// crosses sit at a different height in every strip, so a slow path there adds its delay to EVERY strip's hand-over and
// lengthens the whole dependency chain of a pair (it did: 48 instead of 30 us per strip on a cfg-4 pair)
struct FastValTag { static constexpr bool slow = false; static constexpr bool val = true; };

// chunk c (steps c CH .. c CH + CH-1, rows c CROWS - SKEW .. c CROWS + CROWS-1 over the 32 lanes) touches only valid rows
__device__ __forceinline__ bool interior_chunk(int c, int n) { return c * CROWS >= SKEW && c * CROWS + CROWS <= n; }

// Sakoe-Chiba band in the difference form.  The band |i - j| <= r is closed under diagonal moves, so an admissible cell's
// diagonal predecessor is admissible (or the border) and only two overrides are needed: on the upper edge (j - i == r) the
// "up" predecessor is outside the band, h_in = +inf; on the lower edge (i - j == r) the "left" one is, v_in = +inf.  Their
// transition weights are then exactly 0 (2^-BIG = 0), so E never leaves the band either.  Cells outside the band compute
// finite values nobody uses.  A (chunk, strip) block needs the overrides only if it can contain an edge cell:
__device__ __forceinline__ bool band_clear(int c, int J, int band) {
    const int lo = c * CROWS - SKEW, hi = c * CROWS + CROWS - 1, jl = J * SW, jh = jl + SW - 1;
    return band < 0 || (hi - jl < band && jh - lo < band);
}

// Chunks of strip J that hold at least one admissible row: [cf, cl].  Chunk c covers rows c CROWS - SKEW .. c CROWS +
// CROWS - 1 over the 32 lanes; column j admits rows j - band .. j + band.  Every column has an admissible row because
// band >= |n - m| (checked on the host), so cf <= cl.
__device__ __forceinline__ void band_chunks(int J, int band, int C, int& cf, int& cl) {
    cf = 0; cl = C - 1;
    if (band < 0) return;
    const long long jl = (long long)J * SW, jh = jl + SW - 1;
    if (jl - band > 0) cf = (int)((jl - band) / CROWS);
    cl = (int)min((long long)(C - 1), (jh + band + SKEW) / CROWS);
}

// ------------------------------------------------------------------------------------------------------------------
// prologue, one launch: clear the work counters / progress words / rings, preset the strip-boundary
// columns VS and ES to the sentinel pattern the consumers poll for, and write the scaled copies of the inputs the two
// wavefront kernels read.  Fill regions are multiples of 16 bytes (the workspace layout aligns them to 256).
struct FillJob { uint4* ptr; unsigned long long count16; unsigned word; };
__global__ void prologue_kernel(const FillJob f0, const FillJob f1, const FillJob f2,
                                const float* __restrict__ X, long long nx, const float* __restrict__ Z, long long nz,
                                float s, float* __restrict__ Xs, float* __restrict__ Zs) {
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    const unsigned long long t = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    for (unsigned long long e = t; e < (unsigned long long)(nx + nz); e += stride) {
        if (e < (unsigned long long)nx) Xs[e] = X[e] * s; else Zs[e - nx] = Z[e - nx] * s;
    }
    const FillJob jobs[3] = {f0, f1, f2};
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        const uint4 v = make_uint4(jobs[q].word, jobs[q].word, jobs[q].word, jobs[q].word);
        for (unsigned long long e = t; e < jobs[q].count16; e += stride) __stcs(jobs[q].ptr + e, v);
    }
}

// ------------------------------------------------------------------------------------------------------------------
// forward: eq. 5 in difference form, value by a staircase sum, strip-boundary column to VS, checkpoints to CK.
// Chunks whose 32 x 32 (step, lane) block lies inside the matrix and off this warp's value staircase run the FAST
// step (no bounds or staircase tests, TR steps unrolled between checkpoints, the two rows of a step interleaved); the
// others run the general step.  Both evaluate every cell with the same expressions.
//
// Schedule: a UNIT is FW adjacent strips of one pair (unit u = g N + ps: group-major, so group g+1 of a pair is taken
// long after its group g).  A CTA of FW warps pops units from a global counter and its warps serve a rolling stream of
// strips: strip s of the CTA's k-th unit goes to the warp whose position is (base_k + s) mod FW, base_k = strips of the
// earlier units.  So a strip and the strip it waits on run on the SAME SM (8 consecutive ones on the same scheduler): a
// warp that has caught up with its producer stops competing with it for the MUFU pipe, which is what balances the
// chain; chains that span SMs leave every SM partly idle.
constexpr int UNIT_RING = 16;
struct RollCtl { int popped; int lock; int uid[UNIT_RING]; int seen[32]; };

// the CTA's k-th unit (>= NU: the queue is empty): popped from the global counter by whichever warp needs it first
template <int FW>
__device__ __forceinline__ int pop_unit(RollCtl& ctl, unsigned* counter, const int k, const int NU, const int warp, const int lane) {
    int u = 0;
    if (lane == 0) {
        volatile RollCtl* vc = &ctl;
        while (vc->popped <= k) {
            if (atomicCAS(&ctl.lock, 0, 1) == 0) {
                const int pc = vc->popped;
                if (pc <= k) {
                    for (;;) {                         // ring slot free: every warp has read unit pc - UNIT_RING
                        int mn = vc->seen[0];
                        for (int w2 = 1; w2 < FW; ++w2) mn = min(mn, vc->seen[w2]);
                        if (mn > pc - UNIT_RING) break;
                        __nanosleep(100);
                    }
                    vc->uid[pc % UNIT_RING] = (int)min(atomicAdd(counter, 1u), (unsigned)NU);
                    __threadfence_block();
                    vc->popped = pc + 1;
                }
                __threadfence_block();
                atomicExch(&ctl.lock, 0);
            } else {
                __nanosleep(50);
            }
        }
        __threadfence_block();
        u = vc->uid[k % UNIT_RING];
        vc->seen[warp] = k + 1;
    }
    return __shfl_sync(FULL, u, 0);
}

template <int D, bool CKPT, int FW>
__global__ void __launch_bounds__(FW * 32, (D >= 3 ? 1 : 32 / FW)) forward_kernel(const Params p) {
    extern __shared__ __align__(16) float smem[];
    __shared__ RollCtl ctl;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float* xs0 = smem + warp * fwd_smem_floats<D>();                 // [2][XWIN][D]
    float2* vin_s = reinterpret_cast<float2*>(xs0 + 2 * XWIN * D);   // [CH] (v_in of lane 0 for the step's two rows)
    float2* vout_s = vin_s + 32;                                     // [CH] (v_out of lane 31)
    const int m = p.m;
    const int US = p.unit_strips;                                    // strips per unit, <= FW
    const int NG1 = p.tail_from / US;                                // full-size groups per pair
    const int NG = NG1 + (p.NS - p.tail_from + p.tail_unit - 1) / p.tail_unit, NU = NG * p.N;   // groups per pair, units
    // position of this warp in the rolling stream: consecutive positions share a scheduler (warp id mod 4)
    const int mypos = (warp & 3) * (FW / 4) + (warp >> 2);
    if (threadIdx.x < 32) { ctl.seen[threadIdx.x] = 0; if (threadIdx.x == 0) { ctl.popped = 0; ctl.lock = 0; } }
    __syncthreads();

    int base = 0;                                          // strips of the units before unit k, mod FW
    unsigned in_q = 0, out_q = 0;                          // ring entries consumed from the left / produced, all strips so far
    for (int k = 0;; ++k) {
        const int u = pop_unit<FW>(ctl, p.counters + 0, k, NU, warp, lane);
        if (u >= NU) break;
        const int g = u / p.N, ps = u - g * p.N;
        const int Jg = (g < NG1) ? g * US : p.tail_from + (g - NG1) * p.tail_unit;   // first strip of this unit
        const int S = (g < NG1) ? US : min(p.tail_unit, p.NS - Jg);                    // strips of this unit
        const int sidx = (mypos - base + FW) % FW;
        base = (base + S) % FW;
        if (sidx >= S) continue;
        const int J = Jg + sidx;
        const PairMeta pm = p.pm[ps];
        const int n = pm.n, C = pm.C;
        const int item = ps * p.NS + J;
        const int T = J * 32 + lane;                       // global thread (column group) index
        const int j0 = T * W;
        // Strip-boundary values.  Gradient path (and forward-only calls without rings): one full column per strip, VS.
        // Forward-only with rings (p.ring != null; CKPT == false, no band, uniform units): inside a unit the boundary
        // values of strip sidx go to the warp one position further through a ring of RING_CHUNKS chunks in global
        // memory (entry = value bits | tag << 32, tag = lap + 1; the buffer is zeroed per evaluation); the producer waits
        // when it is a whole ring ahead of what the consumer has taken (ring_prog).  Only the LAST strip of a unit keeps
        // a full column (its consumer is handed out much later): column g of the pair after unit g.  A warp's ring and
        // its counters run on across the units it serves: producer (position q) and consumer (q + 1) see the same
        // sequence of strips, so their cumulative entry counts agree.
        const bool rings = !CKPT && p.ring != nullptr;
        const bool in_ring = rings && sidx > 0, out_ring = rings && sidx + 1 < S;
        const bool out_none = rings && !out_ring && J == p.NS - 1;            // nobody reads the last strip's boundary
        const long long col = rings ? (out_ring ? 0 : g) : J;                 // my output column (when I have one)
        float* VSme = p.VS + pm.vs_off + col * pm.vs_stride + VS_PAD;         // indexed by row
        const float* VSprev = rings ? p.VS + pm.vs_off + (long long)(g - 1) * pm.vs_stride + VS_PAD : VSme - pm.vs_stride;
        float* CKme = p.CK + pm.ck_off + (long long)J * pm.ck_stride;
        if constexpr (CKPT) {
            // The reverse pass polls its message columns ES for a sentinel, as this kernel does VS.  This strip presets
            // the ES column of its own (pair, strip) here: 120 KB of streaming stores per strip next to 4 ms of arithmetic,
            // instead of a 2.8 GB fill in the prologue (0.4 ms on cfg 4) while every SM idles.
            uint4* es = reinterpret_cast<uint4*>(p.ES + pm.vs_off + (long long)J * pm.vs_stride);
            const uint4 sv = make_uint4(SENTINEL, SENTINEL, SENTINEL, SENTINEL);
            for (int q = lane; q < pm.vs_stride / 4; q += 32) __stcs(es + q, sv);
        }
        // ring of the warp at position q of this CTA, and the count of entries that warp has taken from its left neighbour
        // (addresses are rebuilt where they are used: the kernel has no registers to spare)
        auto ring_of = [&](const int q) { return p.ring + ((size_t)blockIdx.x * FW + q) * (RING_ENTRIES * 2); };
        auto prog_of = [&](const int q) { return p.ring_prog + (size_t)blockIdx.x * FW + q; };

        float z[W][D], h[W];
#pragma unroll
        for (int w = 0; w < W; ++w) {
            const int j = j0 + w;
#pragma unroll
            for (int c = 0; c < D; ++c) z[w][c] = (j < m) ? __ldg(p.Zs + (long long)j * D + c) : 0.f;
            h[w] = (j == 0) ? BIG : 0.f;                   // virtual row 0: r_00 = 0, r_0j = inf
        }
        float vp0 = 0.f, vp1 = 0.f;                        // v_out of this lane's last column, rows 2(s-l) and 2(s-l)+1

        // staircase for the value: r_{n,m} = sum of h along row r_h (columns jlo..jhi) + sum of v down one column
        // (rows r_v0+1 .. r_v1) over all threads; see DESIGN.md section 5.4
        const int Tfull = m / W;
        int r_h, r_v0, r_v1, jlo, jhi;
        bool vfirst_sel = false;
        if (Tfull == 0 && T == 0) { r_h = n - 1; jlo = 1; jhi = m - 1; r_v0 = 0; r_v1 = n - 1; vfirst_sel = true; }
        else if (T < Tfull) {
            // staircase rows are ODD rows (the second row of a step) wherever possible: a thread's h[] then holds exactly
            // that row after the step, so the fast path needs no bookkeeping inside its cell loop.  Row n - 1 may be even;
            // it never lies in an interior chunk, so only the general step meets it.
            auto rho = [&](const long long Tq) { return min(n - 1, (int)min((long long)(n - 1), Tq * W * n / m) | 1); };
            const int rho_prev = (T == 0) ? 0 : rho(T);
            const int rho_cur = (T == Tfull - 1) ? n - 1 : rho(T + 1);
            r_h = rho_prev; jlo = max(1, j0); jhi = j0 + W - 1; r_v0 = rho_prev; r_v1 = rho_cur;
        } else { r_h = n - 1; jlo = j0; jhi = m - 1; r_v0 = r_v1 = n - 1; }
        float vacc = 0.f, hsum = 0.f;
        // chunks that hold a staircase row of some lane of this warp (row i of lane l is visited at step i/2 + l)
        const int c_v0 = (__reduce_min_sync(FULL, min(r_h, r_v0)) / RP) / CH;
        const int c_v1 = (__reduce_max_sync(FULL, max(r_h, r_v1)) / RP + 31) / CH;

        const float* xs_lane = xs0;                        // set per chunk
        const int band = p.band;
        // general row: all W cells of row i, plus this thread's piece of the value staircase
        auto slow_row = [&](const int i, const XRow<D>& x, float& v) {
            float vfirst = 0.f, dummy0, dummy1;
#pragma unroll
            for (int w = 0; w < W; ++w) {
                float tl, acc;
                sqdist2<D>(x, z[w], tl, acc);
                if (band >= 0) {                           // band edges: the predecessor outside the band counts as +inf
                    if (j0 + w - i == band) h[w] = BIG;
                    if (i - (j0 + w) == band) v = BIG;
                }
                cell<false, (D > 1)>(tl, acc, h[w], v, dummy0, dummy1, D <= 2 && ((((i & 1) ? SDTW_POLY_MASK_B : SDTW_POLY_MASK_A) >> w) & 1));
                if (w == 0) vfirst = v;
            }
            if ((unsigned)(i - r_v0 - 1) < (unsigned)(r_v1 - r_v0)) vacc += vfirst_sel ? vfirst : v;
            if (i == r_h) {
#pragma unroll
                for (int w = 0; w < W; ++w) if (j0 + w >= jlo && j0 + w <= jhi) hsum += h[w];
            }
            if (T == 0 && i == 0) hsum += sqdist<D>(x, z[0]);   // r_11 = D_11
        };
        auto step = [&](const int c, const int t, auto tag) {
            constexpr bool slow = decltype(tag)::slow;
            float va = __shfl_up_sync(FULL, vp0, 1), vb = __shfl_up_sync(FULL, vp1, 1);
            if (lane == 0) { const float2 qv = vin_s[t]; va = qv.x; vb = qv.y; }
            XRow<D> xa, xb;
            load_x2<D>(xs_lane, 2 * t, xa, xb);
            if constexpr (!slow) {
                constexpr bool val = decltype(tag)::val;
                const int i0 = RP * (c * CH + t - lane);   // used by the staircase bookkeeping only
                float dummy0, dummy1;
#pragma unroll
                for (int w = 0; w < W; ++w) {              // cell (A, w+1) and cell (A+1, w) are independent
                    float tl, acc;
                    sqdist2<D>(xa, z[w], tl, acc);
                    cell<false, (D > 1)>(tl, acc, h[w], va, dummy0, dummy1, D <= 2 && ((SDTW_POLY_MASK_A >> w) & 1));
                    sqdist2<D>(xb, z[w], tl, acc);
                    cell<false, (D > 1)>(tl, acc, h[w], vb, dummy0, dummy1, D <= 2 && ((SDTW_POLY_MASK_B >> w) & 1));
                }
                if (val) {                                 // same additions, in the same order, as the general row
                    if ((unsigned)(i0 - r_v0 - 1) < (unsigned)(r_v1 - r_v0)) vacc += va;
                    if ((unsigned)(i0 - r_v0) < (unsigned)(r_v1 - r_v0)) vacc += vb;
                    if (i0 + 1 == r_h) {                   // r_h is odd inside an interior chunk: h[] is that row now
#pragma unroll
                        for (int w = 0; w < W; ++w) if (j0 + w >= jlo && j0 + w <= jhi) hsum += h[w];
                    }
                }
                vp0 = va; vp1 = vb;
            } else {
                const int i0 = RP * (c * CH + t - lane);
                if ((unsigned)i0 < (unsigned)n) { slow_row(i0, xa, va); vp0 = va; }
                if ((unsigned)(i0 + 1) < (unsigned)n) { slow_row(i0 + 1, xb, vb); vp1 = vb; }
            }
            if (lane == 31) vout_s[t] = make_float2(vp0, vp1);
        };
        auto checkpoint = [&](const int idx) {             // state after step idx*TR - 1
            float* ck = CKme + (long long)idx * CK_FLOATS;
#pragma unroll
            for (int g = 0; g < W / 4; ++g)
                __stcs(reinterpret_cast<float4*>(ck) + g * 32 + lane, make_float4(h[4 * g], h[4 * g + 1], h[4 * g + 2], h[4 * g + 3]));
            __stcs(reinterpret_cast<float2*>(ck + W * 32) + lane, make_float2(vp0, vp1));
        };

        // prefetch of chunk 0: the cycle's rows (cp.async) and the left strip's boundary values (registers)
        // band: chunks above / below the band are not swept.  Starting at chunk cf from the zero state is exact: whatever
        // an admissible cell takes from a skipped chunk is an input the band-edge override replaces.
        int cf, cl;
        band_chunks(J, band, C, cf, cl);
        stage_x_async<D>(xs0 + (cf & 1) * XWIN * D, p.Xs, pm.x_off, n, cf, lane);
        const int vlane = (lane < CH) ? lane : 0;          // lanes >= CH duplicate lane 0's poll (CH < 32 only)
        float2 vreg = make_float2(0.f, 0.f);
        bool vbad = false;                                 // vreg is not the published value yet
        // boundary values of rows r, r + 1 (r = c CROWS + 2 vlane) from the left strip: column or ring; rows >= n are never used
        auto load_in = [&](const int c) {
            const int r = c * CROWS + 2 * vlane;
            if (in_ring) {
                const unsigned e = in_q + (unsigned)(c * CH + vlane);
                unsigned long long a, b2;
                ld_relaxed_v2u64(ring_of((mypos + FW - 1) % FW) + (size_t)(e & (RING_ENTRIES - 1)) * 2, a, b2);
                const unsigned tag = e / RING_ENTRIES + 1u;
                vreg = make_float2(__uint_as_float((unsigned)a), __uint_as_float((unsigned)b2));
                vbad = (r < n && (unsigned)(a >> 32) != tag) || (r + 1 < n && (unsigned)(b2 >> 32) != tag);
            } else {
                vreg = ld_relaxed_f2(VSprev + r);
                vbad = (r < n && is_sentinel(vreg.x)) || (r + 1 < n && is_sentinel(vreg.y));
            }
        };
        if (J > 0) load_in(cf);
        unsigned cons_seen = 0;                            // my consumer's progress as last read (rings)

        for (int c = cf; c <= cl; ++c) {
            const int rbase = c * CROWS + 2 * vlane;       // lane 0 works on rows rbase, rbase + 1 at step `vlane`
            if (J > 0) {                                   // valid = the left strip has published these rows
                if (__any_sync(FULL, vbad)) {
                    for (;;) {
                        if (vbad) load_in(c);
                        if (!__any_sync(FULL, vbad)) break;
                        __nanosleep(100);
                    }
                }
            } else {
                vreg = make_float2(rbase == 0 ? BIG : 0.f, 0.f);
            }
            cp_async_wait_all();
            if (lane < CH) vin_s[lane] = vreg;
            __syncwarp();
            if (in_ring && lane == 0) st_relaxed_u32(prog_of(mypos), in_q + (unsigned)((c + 1) * CH));   // chunk c taken
            if (out_ring && lane == 0) cons_seen = ld_relaxed_u32(prog_of((mypos + 1) % FW));           // looked at below
            if (c + 1 <= cl) {                             // prefetch of chunk c + 1 (the other x buffer)
                stage_x_async<D>(xs0 + ((c + 1) & 1) * XWIN * D, p.Xs, pm.x_off, n, c + 1, lane);
                if (J > 0) load_in(c + 1);
            }
            xs_lane = xs0 + (c & 1) * XWIN * D + (XPAD - 2 * lane) * D;    // rows of step t: xs_lane[2t], [2t+1]
            const bool inside = interior_chunk(c, n) && band_clear(c, J, band);
            if (inside && (c < c_v0 || c > c_v1)) {
#pragma unroll 1
                for (int b = 0; b < CH / TR; ++b) {
#pragma unroll
                    for (int u = 0; u < TR; ++u) step(c, b * TR + u, FastTag{});
                    if (CKPT) checkpoint(c * (CH / TR) + b + 1);
                }
            } else if (inside && Tfull > 0) {              // on this warp's value staircase
#pragma unroll 1
                for (int b = 0; b < CH / TR; ++b) {
#pragma unroll
                    for (int u = 0; u < TR; ++u) step(c, b * TR + u, FastValTag{});
                    if (CKPT) checkpoint(c * (CH / TR) + b + 1);
                }
            } else {
#pragma unroll 1
                for (int t = 0; t < CH; ++t) {
                    step(c, t, SlowTag{});
                    if (CKPT && ((t + 1) & (TR - 1)) == 0) checkpoint((c * CH + t + 1) / TR);
                }
            }
            __syncwarp();
            // lane 31 worked on rows c CROWS - SKEW + 2t (+1) at step t
            if (out_ring) {
                // entry of rows (r, r + 1): out_base + r / 2.  The highest entry of this chunk reuses the slot of the entry
                // RING_ENTRIES below it (an entry of this strip or of the strip before): my consumer must have taken it
                {
                    const unsigned need = out_q + (unsigned)((c - RING_CHUNKS + 1) * CH);   // cumulative; wraps like the counters
                    unsigned seen = __shfl_sync(FULL, cons_seen, 0);
                    while ((int)(seen - need) < 0) {
                        __nanosleep(64);
                        if (lane == 0) cons_seen = ld_relaxed_u32(prog_of((mypos + 1) % FW));
                        seen = __shfl_sync(FULL, cons_seen, 0);
                    }
                }
                const int q = c * CH - (SKEW / 2) + lane;               // r / 2 for r = c CROWS - SKEW + 2 lane
                if (lane < CH && q >= 0) {
                    const unsigned e = out_q + (unsigned)q;
                    const unsigned long long tag = (unsigned long long)(e / RING_ENTRIES + 1u) << 32;
                    const float2 vo = vout_s[lane];
                    st_relaxed_v2u64(ring_of(mypos) + (size_t)(e & (RING_ENTRIES - 1)) * 2, tag | __float_as_uint(vo.x), tag | __float_as_uint(vo.y));
                }
            } else if (!out_none) {
                if (lane < CH) st_relaxed_f2(VSme + c * CROWS - SKEW + 2 * lane, vout_s[lane]);
            }
        }
        if (in_ring) in_q += (unsigned)(C * CH);
        if (out_ring) out_q += (unsigned)(C * CH);
        if (cl < C - 1) {
            // the right strip's last chunks (its band ends SW rows lower) still poll rows this strip never reaches: they
            // feed only cells outside the band or overridden inputs, so publish zeros for them
            const int r0 = (cl + 1) * CROWS - SKEW, r1 = min(C, cl + 2 + SW / CROWS + 1) * CROWS;
            for (int r = r0 + 2 * lane; r < r1; r += 64) st_relaxed_f2(VSme + r, make_float2(0.f, 0.f));
        }
        // value partial of this item
        double part = (double)hsum + (double)vacc;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(FULL, part, o);
        if (lane == 0) p.VP[item] = part;
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------------------------------
// reverse: restore checkpoint, recompute TR steps (weights -> smem), E recurrence backwards, gradient contraction.
// The flow of E out of a cell is split with fused multiply-adds: with (wu, wl) the cell's "up" / "left" weights,
//   into (i-1, j): E wu      into (i, j-1): E wl      into (i-1, j-1): E - E wu - E wl   (mass conserving)
template <int D>
__global__ void __launch_bounds__(WARPS * 32) backward_kernel(const Params p) {
    extern __shared__ __align__(16) float smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float* base = smem + warp * bwd_smem_floats<D>();
    float2* stash = reinterpret_cast<float2*>(base) + lane;     // [TR][RP][W][32] (+ lane)
    float* xs = base + TR * RP * W * 32 * 2;                    // [XWIN][D]
    float2* vin_s = reinterpret_cast<float2*>(xs + XWIN * D);   // [CH]
    float2* ein_s = vin_s + 32;                                 // [CH] messages into lane 31: (.x row 2(s-31), .y the next)
    float2* eout_s = ein_s + 32;                                // [CH] messages out of lane 0
    const float* xs_lane = xs + (XPAD - 2 * lane) * D;
    const int m = p.m;
    constexpr int BPC = CH / TR;

    for (;;) {
        unsigned q = 0;
        if (lane == 0) q = atomicAdd(p.counters + 1, 1u);
        q = __shfl_sync(FULL, q, 0);
        if (q >= p.num_items) break;
        const int Jr = q / p.N, ps = q - Jr * p.N;
        const int J = p.NS - 1 - Jr;                          // right-most strip first
        const PairMeta pm = p.pm[ps];
        const int n = pm.n, C = pm.C;
        const int item = ps * p.NS + J;
        const int j0 = (J * 32 + lane) * W;
        const bool has_right = (J < p.NS - 1);
        const int band = p.band;
        int cf, cl;                                           // chunks of this strip with rows inside the band
        band_chunks(J, band, C, cf, cl);
        const int bfirst = cf * BPC;
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
            A[w] = (j == m - 1) ? 1.f : 0.f;                  // E[n+1][m+1] = 1 flows into cell (n, m)
            h[w] = 0.f;
        }
        float vp0 = 0.f, vp1 = 0.f;
        float msg0_prev = 0.f, msg1_prev = 0.f, cdf_prev = 0.f;

        // prefetch of the next checkpoint to restore
        float4 ph[W / 4]; float2 pv = make_float2(0.f, 0.f);
        auto prefetch = [&](int bidx) {
            if (bidx > bfirst) {                              // block bfirst starts from the zero state, not a checkpoint
                const float* ck = CKme + (long long)bidx * CK_FLOATS;
#pragma unroll
                for (int gq = 0; gq < W / 4; ++gq) ph[gq] = __ldcs(reinterpret_cast<const float4*>(ck) + gq * 32 + lane);
                pv = __ldcs(reinterpret_cast<const float2*>(ck + W * 32) + lane);
            }
        };
        prefetch((cl + 1) * BPC - 1);

        // one row of the recompute, keeping the transition weights
        auto rec_row = [&](const int i, const XRow<D>& x, float& v, const int slot) {
#pragma unroll
            for (int w = 0; w < W; ++w) {
                float tl, acc, wu, wl;
                sqdist2<D>(x, z[w], tl, acc);
                if (band >= 0) {                              // band edges, as in the forward kernel
                    if (j0 + w - i == band) h[w] = BIG;
                    if (i - (j0 + w) == band) v = BIG;
                }
                cell<true, (D > 1)>(tl, acc, h[w], v, wu, wl);
                stash[(slot * W + w) * 32] = make_float2(wu, wl);
            }
        };
        // recompute step t of the chunk (u = t - t0 within the block)
        auto recompute = [&](const int c, const int t, const int u, auto tag) {
            constexpr bool slow = decltype(tag)::slow;
            float va = __shfl_up_sync(FULL, vp0, 1), vb = __shfl_up_sync(FULL, vp1, 1);
            if (lane == 0) { const float2 qv = vin_s[t]; va = qv.x; vb = qv.y; }
            XRow<D> xa, xb;
            load_x2<D>(xs_lane, 2 * t, xa, xb);
            if constexpr (!slow) {
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
            } else {
                const int i0 = RP * (c * CH + t - lane);
                if ((unsigned)i0 < (unsigned)n) { rec_row(i0, xa, va, u * RP + 0); vp0 = va; }
                if ((unsigned)(i0 + 1) < (unsigned)n) { rec_row(i0 + 1, xb, vb, u * RP + 1); vp1 = vb; }
            }
        };
        // E recurrence of one row, right to left: E_in = flow into the last column's cell from the right neighbour;
        // returns the left flow out of column 0 (cl) and the diagonal share of column 0 (cd)
        auto e_row = [&](const XRow<D>& x, const float e_in, const int slot, float& cl, float& cd) {
            float E = A[W - 1] + e_in;
            float cd_right = 0.f;
#pragma unroll
            for (int w = W - 1; w >= 0; --w) {
                const float2 wt = stash[(slot * W + w) * 32];
#pragma unroll
                for (int ch = 0; ch < D; ++ch) g[w][ch] = fmaf(E, z[w][ch] - x.c[ch], g[w][ch]);
                const float Anew = fmaf(E, wt.x, cd_right);       // into (i-1, j): from (i, j) and, diagonally, (i, j+1)
                cd_right = fmaf(-E, wt.y, fmaf(-E, wt.x, E));     // diagonal share of this cell
                if (w > 0) E = fmaf(E, wt.y, A[w - 1]); else cl = E * wt.y;
                A[w] = Anew;
            }
            cd = cd_right;
        };
        // E recurrence for the same step, backwards (probability flow, mass conserving): row 2(s-l)+1, then row 2(s-l)
        auto eflow = [&](const int c, const int t, const int u, auto tag) {
            constexpr bool slow = decltype(tag)::slow;
            float in0 = __shfl_down_sync(FULL, msg0_prev, 1), in1 = __shfl_down_sync(FULL, msg1_prev, 1);
            if (lane == 31) { const float2 qe = ein_s[t]; in0 = qe.x; in1 = qe.y; }
            XRow<D> xa, xb;
            load_x2<D>(xs_lane, 2 * t, xa, xb);
            const int i0 = RP * (c * CH + t - lane);
            float cd_mid = cdf_prev;                           // row i0+1 missing (i0 + 1 == n): its diagonal share is 0
            if (!slow || (unsigned)(i0 + 1) < (unsigned)n) {
                float cl1, cd1;
                e_row(xb, in1, u * RP + 1, cl1, cd1);
                msg1_prev = cl1 + cdf_prev;                    // into the left neighbour's cell (i0+1, j0-1)
                cd_mid = cd1;
            }
            if (!slow || (unsigned)i0 < (unsigned)n) {
                float cl0, cd0;
                e_row(xa, in0, u * RP + 0, cl0, cd0);
                msg0_prev = cl0 + cd_mid;                      // into (i0, j0-1)
                cdf_prev = cd0;
            }
            if (lane == 0) eout_s[t] = make_float2(msg0_prev, msg1_prev);
        };

        // Progress word of an item: chunks completed from the top (C - c after chunk c); when the item is done,
        // FIN | z: every message of its chunks [0, z) is an implicit +0 (they were never visited).
        constexpr unsigned FIN = 0x80000000u;
        // Strip-to-strip exchange of the reverse pass, without flags or fences on the way (as in the forward kernel): ES is
        // preset to the sentinel pattern, the right strip writes its messages with relaxed stores, this strip polls the
        // DATA words, one chunk ahead of use.  Only the end of an item is published with a release: its progress word
        // becomes FIN | z, "done, and every message of my chunks [0, z) is an implicit +0 (never written)".
        unsigned finw = 0;                                     // the right strip's progress word as last seen
        auto poll_fin = [&]() {
            if (has_right && !(finw & FIN)) {
                unsigned f = 0;
                if (lane == 0) f = ld_acquire(p.prog_b + item + 1);
                finw = __shfl_sync(FULL, f, 0);
                __syncwarp();                                  // the other lanes reload ES only after lane 0's acquire
            }
        };
        auto load_msg = [&](const int c) {                     // lane t: the message pair of lane 31's step t of chunk c
            const int r = c * CROWS - SKEW + 2 * lane;
            return (has_right && lane < CH && r >= 0) ? ld_relaxed_f2(ESnext + r) : make_float2(0.f, 0.f);
        };
        auto peek_fin = [&]() { return (has_right && lane == 0) ? ld_relaxed_u32(p.prog_b + item + 1) : 0u; };
        float2 ereg = load_msg(cl);
        unsigned freg = peek_fin();                            // prefetched with the messages; a stale value only delays
        int pf = (cl + 1) * BPC - 1;                           // block whose checkpoint (ph, pv) currently holds
        unsigned long long skipped = 0;
        bool terminated = false;
        for (int c = cl; c >= cf; --c) {
            unsigned lbits = __float_as_uint(msg0_prev) | __float_as_uint(msg1_prev) | __float_as_uint(cdf_prev);
#pragma unroll
            for (int w = 0; w < W; ++w) lbits |= __float_as_uint(A[w]);
            const bool local_nz = __any_sync(FULL, lbits != 0u);     // flow already inside this strip
            // lane 31 works on rows c CROWS - SKEW + 2t (+1) at step t; lane t holds its message pair in ereg
            const int erow = c * CROWS - SKEW + 2 * lane;
            float2 ein = ereg;
            if (has_right) {
                bool bad = is_sentinel(ein.x) || is_sentinel(ein.y);
                if (__shfl_sync(FULL, freg, 0) & FIN) poll_fin();        // the right strip is done: make that official (acquire)
                while (__any_sync(FULL, bad)) {
                    // not published yet -- or never will be: the right strip is done and these rows lie in chunks it
                    // did not visit (after the acquire in poll_fin every row it did write is visible)
                    if (bad) {
                        ein = ld_relaxed_f2(ESnext + erow);
                        bad = is_sentinel(ein.x) || is_sentinel(ein.y);
                        if (bad && (finw & FIN) && erow / CROWS < (int)(finw & ~FIN)) { ein = make_float2(0.f, 0.f); bad = false; }
                    }
                    if (__any_sync(FULL, bad)) { __nanosleep(64); poll_fin(); }
                }
            }
            const bool rfin = (finw & FIN) != 0u;
            const int zr = (int)(finw & ~FIN);                 // valid when rfin
            // Early exit: nothing flows inside this strip and nothing will ever arrive from the right (there is no right
            // strip, or it is done and its remaining messages are implicit zeros): every chunk from here down is a skip.
            if (!p.dense_reverse && !local_nz && (!has_right || (rfin && c < zr))) {
                __syncwarp();
                if (lane == 0) st_release(p.prog_b + item, FIN | (unsigned)(c + 1));
                skipped += (unsigned long long)(c - cf + 1);
                terminated = true;
                break;
            }
            if (c > cf) { ereg = load_msg(c - 1); freg = peek_fin(); }   // prefetch for the next chunk
            // Exact skip: every flow that could enter this chunk's cells is +0 (E underflows to zero off the
            // alignment band), so every product and sum below would be +0 and g would not change.
            if (!p.dense_reverse && !local_nz) {
                const unsigned bits = __float_as_uint(ein.x) | __float_as_uint(ein.y);
                if (!__any_sync(FULL, bits != 0u)) {
                    if (J > 0 && lane < CH) st_relaxed_f2(ESme + c * CROWS + 2 * lane, make_float2(0.f, 0.f));
                    ++skipped;
                    continue;
                }
            }
            stage_x_async<D>(xs, p.Xs, pm.x_off, n, c, lane);
            if (lane < CH) {
                const int rbase = c * CROWS + 2 * lane;
                vin_s[lane] = (J > 0) ? __ldcs(reinterpret_cast<const float2*>(VSprev + rbase))
                                      : make_float2(rbase == 0 ? BIG : 0.f, 0.f);
                ein_s[lane] = ein;
            }
            cp_async_wait_all();
            __syncwarp();
            const bool fast = interior_chunk(c, n) && band_clear(c, J, band);
#pragma unroll 1
            for (int b = BPC - 1; b >= 0; --b) {
                const int bidx = c * BPC + b, t0 = b * TR;
                if (bidx == bfirst) {                          // the forward sweep started here from the zero state
#pragma unroll
                    for (int w = 0; w < W; ++w) h[w] = (bidx == 0 && j0 + w == 0) ? BIG : 0.f;
                    vp0 = vp1 = 0.f;
                } else {
                    if (pf != bidx) prefetch(bidx);            // the chunk below was skipped: nothing was prefetched
#pragma unroll
                    for (int gq = 0; gq < W / 4; ++gq) { h[4 * gq] = ph[gq].x; h[4 * gq + 1] = ph[gq].y; h[4 * gq + 2] = ph[gq].z; h[4 * gq + 3] = ph[gq].w; }
                    vp0 = pv.x; vp1 = pv.y;
                }
                prefetch(bidx - 1);
                pf = bidx - 1;
                if (fast) {
#pragma unroll
                    for (int u = 0; u < TR; ++u) recompute(c, t0 + u, u, FastTag{});
#pragma unroll
                    for (int u = TR - 1; u >= 0; --u) eflow(c, t0 + u, u, FastTag{});
                } else {
#pragma unroll 1
                    for (int u = 0; u < TR; ++u) recompute(c, t0 + u, u, SlowTag{});
#pragma unroll 1
                    for (int u = TR - 1; u >= 0; --u) eflow(c, t0 + u, u, SlowTag{});
                }
            }
            __syncwarp();
            // lane 0 worked on rows 64c + 2t (+1) at step t
            if (J > 0 && lane < CH) st_relaxed_f2(ESme + c * CROWS + 2 * lane, eout_s[lane]);
        }
        // done: the chunks below cf (above the band) were never visited, their messages are implicit zeros
        if (!terminated) {
            __syncwarp();
            if (lane == 0) st_release(p.prog_b + item, FIN | (unsigned)cf);
        }
        skipped += (unsigned long long)(C - 1 - cl + cf);
        if (lane == 0 && p.stats) { atomicAdd(p.stats + 0, (unsigned long long)C); atomicAdd(p.stats + 1, skipped); }
        // eq. 6 partial of this pair for this strip's columns, back in natural units
#pragma unroll
        for (int w = 0; w < W; ++w) {
            const int j = j0 + w;
            if (j < m) {
#pragma unroll
                for (int ch = 0; ch < D; ++ch) p.Gk[((long long)ps * m + j) * D + ch] = g[w][ch] * p.gscale;
            }
        }
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------------------------------
// epilogue, one launch.  Last block (if want_values): per-pair values from the item partials in caller order, objective
// (eq. 7: sum_k w_k value_k) by a fixed-shape tree.  Other blocks (if md > 0): G[e] = sum over pairs in schedule order with
// an fp64 accumulator (deterministic, no atomics), optionally fused with the descent step Z <- Z - step G.
__global__ void epilogue_kernel(const double* __restrict__ VP, const PairMeta* __restrict__ pm, const float* __restrict__ wts,
                                int N, int NS, double inv_kappa, int want_values, float* __restrict__ out_values,
                                float* __restrict__ out_objective, double* __restrict__ out_objective64,
                                const float* __restrict__ Gk, long long md, float* __restrict__ out_grad, float* __restrict__ Z,
                                float step) {
    __shared__ double red[256];
    if (want_values && blockIdx.x == gridDim.x - 1) {
        double local = 0.0;
        for (int ps = threadIdx.x; ps < N; ps += blockDim.x) {
            double s = 0.0;
            for (int J = 0; J < NS; ++J) s += VP[(long long)ps * NS + J];
            s *= inv_kappa;
            if (out_values) out_values[pm[ps].k] = (float)s;
            local += wts ? (double)wts[ps] * s : s;
        }
        red[threadIdx.x] = local;
        __syncthreads();
        for (int o = blockDim.x / 2; o > 0; o >>= 1) {
            if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
            __syncthreads();
        }
        if (threadIdx.x == 0 && out_objective) *out_objective = (float)red[0];
        if (threadIdx.x == 0 && out_objective64) *out_objective64 = red[0];
        return;
    }
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= md) return;
    double acc = 0.0;
    if (wts) { for (int ps = 0; ps < N; ++ps) acc += (double)wts[ps] * (double)Gk[(long long)ps * md + e]; }
    else     { for (int ps = 0; ps < N; ++ps) acc += (double)Gk[(long long)ps * md + e]; }
    const float gsum = (float)acc;
    if (out_grad) out_grad[e] = gsum;
    if (Z) Z[e] = Z[e] - step * gsum;
}

// line-search helpers: the trial point Zt = Z - t G, and ||G||^2 by a fixed-shape tree (one block; deterministic)
__global__ void trial_point_kernel(float* __restrict__ Zt, const float* __restrict__ Z, const float* __restrict__ G,
                                   long long count, float t) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < count) Zt[e] = Z[e] - t * G[e];
}
__global__ void sqnorm_kernel(const float* __restrict__ G, long long count, double* __restrict__ out) {
    __shared__ double red[1024];
    double acc = 0.0;
    for (long long e = threadIdx.x; e < count; e += blockDim.x) acc += (double)G[e] * (double)G[e];
    red[threadIdx.x] = acc;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = red[0];
}

// L-BFGS helpers (sdtw_barycenter_lbfgs): a . b by a fixed-shape tree in float64 (one block; deterministic), and the
// vector updates of the two-loop recursion, in float32 with a float64 scalar rounded once
__global__ void dot_kernel(const float* __restrict__ a, const float* __restrict__ b, long long count, double* __restrict__ out) {
    __shared__ double red[1024];
    double acc = 0.0;
    for (long long e = threadIdx.x; e < count; e += blockDim.x) acc += (double)a[e] * (double)b[e];
    red[threadIdx.x] = acc;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = red[0];
}
// y = a x + b y  (b = 0: y = a x, y need not be initialised).  x may BE y (the in-place scalings of the L-BFGS
// recursion), so neither pointer is __restrict__: every thread reads element e before it writes it.
__global__ void axpby_kernel(float* y, const float* x, long long count, float a, float b) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < count) y[e] = (b == 0.f) ? a * x[e] : fmaf(a, x[e], b * y[e]);
}
// out = a - b
__global__ void diff_kernel(float* __restrict__ out, const float* __restrict__ a, const float* __restrict__ b, long long count) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < count) out[e] = a[e] - b[e];
}

__global__ void gd_update_kernel(float* __restrict__ Z, const float* __restrict__ G, long long count, float step) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < count) Z[e] = Z[e] - step * G[e];
}

}  // namespace sdtw
