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
// warp.  Lane l works on row (step - l): the anti-diagonal wavefront.  Neighbouring lanes exchange one value per step
// by warp shuffle; neighbouring strips exchange the strip-boundary column through global memory (VS forward, ES
// reverse) with a release/acquire progress counter per item.  Every TR steps the forward kernel checkpoints the warp
// state (h[W] + the value in flight) to HBM; the reverse kernel restores a checkpoint, recomputes TR steps keeping the
// transition weights in shared memory, then runs the E recurrence over those TR steps backwards, accumulating the
// gradient contraction of eq. 6 in registers.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sdtw {

constexpr int W = 4;            // columns per thread
constexpr int SW = 32 * W;      // columns per strip (work item)
constexpr int CH = 32;          // steps per chunk (granularity of the strip-boundary exchange)
constexpr int TR = 8;           // steps between checkpoints (= rows recomputed per reverse block)
constexpr int WARPS = 4;        // warps per CTA (each warp is an independent agent)
constexpr int CK_FLOATS = 32 * (W + 1);  // floats per checkpoint record
constexpr float BIG = 1.0e30f;  // stands for the +inf border of eq. 5
constexpr unsigned FULL = 0xffffffffu;

struct PairMeta {   // one per pair, in schedule order (longest first)
    long long x_off;      // first row of this cycle in X_concat
    long long vs_off;     // float offset of strip 0's boundary column in VS / ES; strip stride = vs_stride
    long long ck_off;     // float offset of strip 0's checkpoints; strip stride = ck_stride
    long long ck_stride;
    int vs_stride;
    int n;                // rows of this cycle
    int k;                // caller's pair index
    int C;                // chunks = ceil((n + 31) / CH)
};

struct Params {
    const float* Z;
    const float* X;
    const PairMeta* pm;
    unsigned* counters;   // [0] forward work queue, [1] reverse work queue
    unsigned* prog_f;     // [N * NS] chunks completed by each forward item
    unsigned* prog_b;     // [N * NS] chunks completed by each reverse item
    float* VS;            // strip-boundary v columns, indexed by producer step
    float* ES;            // strip-boundary E messages, indexed by row (32 floats of front padding per strip)
    float* CK;            // checkpoints
    double* VP;           // [N * NS] per-item partial of the value (staircase sum), scaled units
    float* Gk;            // [N][m][D] per-pair gradient partials
    int m, N, NS;
    unsigned num_items;
    unsigned long long* stats;  // [0] reverse chunks visited, [1] reverse chunks skipped (instrumentation; may be null)
    int dense_reverse;    // 1: never skip a reverse chunk (for measurement / validation of the exact skip)
    float sqrtk;          // sqrt(1 / (gamma ln 2))
    float gscale;         // 2 / sqrtk
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

// shared memory per warp (floats)
template <int D> __host__ __device__ constexpr int fwd_smem_floats() { return 64 * D + 64; }
template <int D> __host__ __device__ constexpr int bwd_smem_floats() { return TR * W * 32 * 2 + 64 * D + 96; }

template <int D> struct XRow { float c[D]; };

template <int D>
__device__ __forceinline__ XRow<D> load_x(const float* xs, int e) {
    XRow<D> r;
    if constexpr (D == 4) {
        float4 t = *reinterpret_cast<const float4*>(xs + e * 4);
        r.c[0] = t.x; r.c[1] = t.y; r.c[2] = t.z; r.c[3] = t.w;
    } else if constexpr (D == 2) {
        float2 t = *reinterpret_cast<const float2*>(xs + e * 2);
        r.c[0] = t.x; r.c[1] = t.y;
    } else {
#pragma unroll
        for (int c = 0; c < D; ++c) r.c[c] = xs[e * D + c];
    }
    return r;
}

// stage rows [c*CH - 32, c*CH + 32) of the (scaled) cycle into xs[64][D]; rows outside [0, n) read as 0
template <int D>
__device__ __forceinline__ void stage_x(float* xs, const float* __restrict__ X, long long x_off, int n, int c, int lane,
                                        float sqrtk) {
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        const int e = lane + 32 * half;
        const int r = c * CH - 32 + e;
        const bool ok = (unsigned)r < (unsigned)n;
#pragma unroll
        for (int ch = 0; ch < D; ++ch) xs[e * D + ch] = ok ? __ldg(X + (x_off + r) * D + ch) * sqrtk : 0.f;
    }
}

// ------------------------------------------------------------------------------------------------------------------
// one cell of the difference-form recurrence.  v is v_in on entry and v_out on return; h is h_in / h_out.
// t2 is the SQUARED cost input: the cell cost is D = sum_c t_c^2, passed as (t_last, acc) with D = t_last^2 + acc so
// that the last square fuses with the subtraction of the log (one FFMA).
// With a = mn - h_in, b = mn - v_in (mn = min(0, h_in, v_in); one of 0, a, b is exactly 0) the three soft-min terms are
// 2^mn (diagonal), 2^a ("up"), 2^b ("left"); sorted, they are 1, e1 = 2^-|min(h,v)| and e2 = 2^min(a,b).
// STASH: also emit the weights (w_up, w_left) of this cell's "up" and "left" predecessors.
__device__ __forceinline__ float min3(float a, float b, float c) {
    float r; asm("min.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r;
}
template <bool STASH, bool HASACC>
__device__ __forceinline__ void cell(float t_last, float acc, float& h, float& v, float& wu, float& wl) {
    const float hin = h, vin = v;
    const float mn = min3(hin, vin, 0.f);
    const float p = fminf(hin, vin);
    const float a = mn - hin, b = mn - vin;
    const float e1 = ex2_approx(-fabsf(p));     // p >= 0: the min(h,v) term;  p < 0: the diagonal term
    const float e2 = ex2_approx(fminf(a, b));   // the max(h,v) term
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

struct FastTag { static constexpr bool slow = false; };
struct SlowTag { static constexpr bool slow = true; };

// chunk c (steps 32c .. 32c+31, rows 32c-31 .. 32c+31 over the 32 lanes) touches only valid rows
__device__ __forceinline__ bool interior_chunk(int c, int n) { return c >= 1 && c * CH + CH <= n; }

// ------------------------------------------------------------------------------------------------------------------
// forward: eq. 5 in difference form, value by a staircase sum, strip-boundary column to VS, checkpoints to CK.
// Chunks whose 32 x 32 (step, lane) block lies inside the matrix and off this warp's value staircase run the FAST
// step (no bounds or staircase tests, 8 steps unrolled between checkpoints); the others run the general step.  Both
// evaluate every cell with the same expressions.
template <int D, bool CKPT>
__global__ void __launch_bounds__(WARPS * 32) forward_kernel(const Params p) {
    extern __shared__ __align__(16) float smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float* xs = smem + warp * fwd_smem_floats<D>();
    float* vin_s = xs + 64 * D;
    float* vout_s = vin_s + 32;
    const float* xs_lane = xs + (32 - lane) * D;           // row (c*CH + t - lane) of the staged window is xs_lane[t*D ..]
    const int m = p.m;

    for (;;) {
        unsigned q = 0;
        if (lane == 0) q = atomicAdd(p.counters + 0, 1u);
        q = __shfl_sync(FULL, q, 0);
        if (q >= p.num_items) break;
        const int J = q / p.N, ps = q - J * p.N;          // strip-major order: all pairs' strip 0 first
        const PairMeta pm = p.pm[ps];
        const int n = pm.n, C = pm.C;
        const int item = ps * p.NS + J;
        const int T = J * 32 + lane;                       // global thread (column group) index
        const int j0 = T * W;
        float* VSme = p.VS + pm.vs_off + (long long)J * pm.vs_stride;
        const float* VSprev = VSme - pm.vs_stride;
        float* CKme = p.CK + pm.ck_off + (long long)J * pm.ck_stride;

        float z[W][D], h[W];
#pragma unroll
        for (int w = 0; w < W; ++w) {
            const int j = j0 + w;
#pragma unroll
            for (int c = 0; c < D; ++c) z[w][c] = (j < m) ? __ldg(p.Z + (long long)j * D + c) * p.sqrtk : 0.f;
            h[w] = (j == 0) ? BIG : 0.f;                   // virtual row 0: r_00 = 0, r_0j = inf
        }
        float vprev = 0.f;

        // staircase for the value: r_{n,m} = sum of h along row r_h (columns jlo..jhi) + sum of v down one column
        // (rows r_v0+1 .. r_v1) over all threads; see DESIGN.md section 5.4
        const int Tfull = m / W;
        int r_h, r_v0, r_v1, jlo, jhi;
        bool vfirst_sel = false;
        if (Tfull == 0 && T == 0) { r_h = n - 1; jlo = 1; jhi = m - 1; r_v0 = 0; r_v1 = n - 1; vfirst_sel = true; }
        else if (T < Tfull) {
            const int rho_prev = (T == 0) ? 0 : (int)min((long long)(n - 1), (long long)T * W * n / m);
            const int rho_cur = (T == Tfull - 1) ? n - 1 : (int)min((long long)(n - 1), (long long)(T + 1) * W * n / m);
            r_h = rho_prev; jlo = max(1, j0); jhi = j0 + W - 1; r_v0 = rho_prev; r_v1 = rho_cur;
        } else { r_h = n - 1; jlo = j0; jhi = m - 1; r_v0 = r_v1 = n - 1; }
        float vacc = 0.f, hsum = 0.f;
        // chunks that hold a staircase row of some lane of this warp (row i of lane l is visited at step i + l)
        const int c_v0 = __reduce_min_sync(FULL, min(r_h, r_v0)) / CH;
        const int c_v1 = (__reduce_max_sync(FULL, max(r_h, r_v1)) + 31) / CH;

        auto step = [&](const int c, const int t, auto tag) {
            constexpr bool slow = decltype(tag)::slow;
            float v = __shfl_up_sync(FULL, vprev, 1);
            if (lane == 0) v = vin_s[t];
            const int i = c * CH + t - lane;
            if (!slow || (unsigned)i < (unsigned)n) {
                const XRow<D> x = load_x<D>(xs_lane, t);
                float vfirst = 0.f, dummy0, dummy1;
#pragma unroll
                for (int w = 0; w < W; ++w) {
                    float tl, acc;
                    sqdist2<D>(x, z[w], tl, acc);
                    cell<false, (D > 1)>(tl, acc, h[w], v, dummy0, dummy1);
                    if (slow && w == 0) vfirst = v;
                }
                vprev = v;
                if constexpr (slow) {
                    if ((unsigned)(i - r_v0 - 1) < (unsigned)(r_v1 - r_v0)) vacc += vfirst_sel ? vfirst : v;
                    if (i == r_h) {
#pragma unroll
                        for (int w = 0; w < W; ++w) if (j0 + w >= jlo && j0 + w <= jhi) hsum += h[w];
                    }
                    if (T == 0 && i == 0) hsum += sqdist<D>(x, z[0]);   // r_11 = D_11
                }
            }
            if (lane == 31) vout_s[t] = vprev;
        };
        auto checkpoint = [&](const int idx) {             // state after step idx*TR - 1
            float* ck = CKme + (long long)idx * CK_FLOATS;
#pragma unroll
            for (int g = 0; g < W / 4; ++g)
                reinterpret_cast<float4*>(ck)[g * 32 + lane] = make_float4(h[4 * g], h[4 * g + 1], h[4 * g + 2], h[4 * g + 3]);
            ck[W * 32 + lane] = vprev;
        };

        unsigned seen = 0;
        for (int c = 0; c < C; ++c) {
            if (J > 0) {                                   // wait until the left strip has published what this chunk reads
                const unsigned need = (unsigned)min(c + 2, C);
                while (seen < need) { seen = ld_acquire(p.prog_f + item - 1); if (seen < need) __nanosleep(128); }
            }
            {
                const int s = c * CH + lane;               // lane 0 works on row s at step s
                vin_s[lane] = (J > 0) ? VSprev[s + 31] : ((s == 0) ? BIG : 0.f);
                stage_x<D>(xs, p.X, pm.x_off, n, c, lane, p.sqrtk);
            }
            __syncwarp();
            if (interior_chunk(c, n) && (c < c_v0 || c > c_v1)) {
#pragma unroll 1
                for (int b = 0; b < CH / TR; ++b) {
#pragma unroll
                    for (int u = 0; u < TR; ++u) step(c, b * TR + u, FastTag{});
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
            VSme[c * CH + lane] = vout_s[lane];
            __syncwarp();                                  // orders every lane's VS store before lane 0's release
            if (lane == 0) st_release(p.prog_f + item, (unsigned)(c + 1));
        }
        // value partial of this item
        double part = (double)hsum + (double)vacc;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(FULL, part, o);
        if (lane == 0) p.VP[item] = part;
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
    float2* stash = reinterpret_cast<float2*>(base) + lane;     // [TR][W][32] (+ lane)
    float* xs = base + TR * W * 32 * 2;
    float* vin_s = xs + 64 * D;
    float* ein_s = vin_s + 32;
    float* eout_s = ein_s + 32;
    const float* xs_lane = xs + (32 - lane) * D;
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
        const float* VSprev = p.VS + pm.vs_off + (long long)(J - 1) * pm.vs_stride;
        float* ESme = p.ES + pm.vs_off + (long long)J * pm.vs_stride + 32;       // 32 floats of front padding
        const float* ESnext = ESme + pm.vs_stride;
        const float* CKme = p.CK + pm.ck_off + (long long)J * pm.ck_stride;

        float z[W][D], g[W][D], A[W], h[W];
#pragma unroll
        for (int w = 0; w < W; ++w) {
            const int j = j0 + w;
#pragma unroll
            for (int c = 0; c < D; ++c) { z[w][c] = (j < m) ? __ldg(p.Z + (long long)j * D + c) * p.sqrtk : 0.f; g[w][c] = 0.f; }
            A[w] = (j == m - 1) ? 1.f : 0.f;                  // E[n+1][m+1] = 1 flows into cell (n, m)
        }
        float vprev = 0.f, msg_prev = 0.f, cdf_prev = 0.f;

        // prefetch of the next checkpoint to restore
        float4 ph[W / 4]; float pv = 0.f;
        auto prefetch = [&](int bidx) {
            if (bidx >= 1) {
                const float* ck = CKme + (long long)bidx * CK_FLOATS;
#pragma unroll
                for (int gq = 0; gq < W / 4; ++gq) ph[gq] = __ldcs(reinterpret_cast<const float4*>(ck) + gq * 32 + lane);
                pv = __ldcs(ck + W * 32 + lane);
            }
        };
        prefetch(C * BPC - 1);

        // recompute step t of the chunk (u = t - t0 within the block), keeping the transition weights
        auto recompute = [&](const int c, const int t, const int u, auto tag) {
            constexpr bool slow = decltype(tag)::slow;
            float v = __shfl_up_sync(FULL, vprev, 1);
            if (lane == 0) v = vin_s[t];
            const int i = c * CH + t - lane;
            if (!slow || (unsigned)i < (unsigned)n) {
                const XRow<D> x = load_x<D>(xs_lane, t);
#pragma unroll
                for (int w = 0; w < W; ++w) {
                    float tl, acc, wu, wl;
                    sqdist2<D>(x, z[w], tl, acc);
                    cell<true, (D > 1)>(tl, acc, h[w], v, wu, wl);
                    stash[(u * W + w) * 32] = make_float2(wu, wl);
                }
                vprev = v;
            }
        };
        // E recurrence for the same step, backwards (probability flow, mass conserving)
        auto eflow = [&](const int c, const int t, const int u, auto tag) {
            constexpr bool slow = decltype(tag)::slow;
            float msg_in = __shfl_down_sync(FULL, msg_prev, 1);
            if (lane == 31) msg_in = ein_s[t];
            const int i = c * CH + t - lane;
            if (!slow || (unsigned)i < (unsigned)n) {
                const XRow<D> x = load_x<D>(xs_lane, t);
                float E = A[W - 1] + msg_in;
                float cd_right = 0.f, cl_out = 0.f;
#pragma unroll
                for (int w = W - 1; w >= 0; --w) {
                    const float2 wt = stash[(u * W + w) * 32];
#pragma unroll
                    for (int ch = 0; ch < D; ++ch) g[w][ch] = fmaf(E, z[w][ch] - x.c[ch], g[w][ch]);
                    const float Anew = fmaf(E, wt.x, cd_right);       // into (i-1, j): from (i, j) and, diagonally, (i, j+1)
                    cd_right = fmaf(-E, wt.y, fmaf(-E, wt.x, E));     // diagonal share of this cell
                    if (w > 0) E = fmaf(E, wt.y, A[w - 1]); else cl_out = E * wt.y;
                    A[w] = Anew;
                }
                msg_prev = cl_out + cdf_prev;                // flow into the left neighbour's cell (i, j0-1)
                cdf_prev = cd_right;
            }
            if (lane == 0) eout_s[t] = msg_prev;
        };

        unsigned seen = 0;
        int pf = C * BPC - 1;                                  // block whose checkpoint (ph, pv) currently holds
        unsigned long long skipped = 0;
        for (int c = C - 1; c >= 0; --c) {
            if (has_right) {                                   // right strip must have finished chunks >= max(c-1, 0)
                const unsigned need = (unsigned)(C - max(c - 1, 0));
                while (seen < need) { seen = ld_acquire(p.prog_b + item + 1); if (seen < need) __nanosleep(64); }
            }
            const int s = c * CH + lane;
            const float ein = has_right ? ESnext[s - 31] : 0.f;   // lane 31 works on row s - 31 at step s
            // Exact skip: every flow that could enter this chunk's cells is +0 (E underflows to zero off the
            // alignment band), so every product and sum below would be +0 and g would not change.
            if (!p.dense_reverse) {
                unsigned bits = __float_as_uint(ein) | __float_as_uint(msg_prev) | __float_as_uint(cdf_prev);
#pragma unroll
                for (int w = 0; w < W; ++w) bits |= __float_as_uint(A[w]);
                if (!__any_sync(FULL, bits != 0u)) {
                    if (J > 0) ESme[c * CH + lane] = 0.f;
                    __syncwarp();
                    if (lane == 0) st_release(p.prog_b + item, (unsigned)(C - c));
                    ++skipped;
                    continue;
                }
            }
            vin_s[lane] = (J > 0) ? __ldcs(VSprev + s + 31) : ((s == 0) ? BIG : 0.f);
            ein_s[lane] = ein;
            stage_x<D>(xs, p.X, pm.x_off, n, c, lane, p.sqrtk);
            __syncwarp();
            const bool fast = interior_chunk(c, n);
#pragma unroll 1
            for (int b = BPC - 1; b >= 0; --b) {
                const int bidx = c * BPC + b, t0 = b * TR;
                if (bidx == 0) {
#pragma unroll
                    for (int w = 0; w < W; ++w) h[w] = (j0 + w == 0) ? BIG : 0.f;
                    vprev = 0.f;
                } else {
                    if (pf != bidx) prefetch(bidx);            // the chunk below was skipped: nothing was prefetched
#pragma unroll
                    for (int gq = 0; gq < W / 4; ++gq) { h[4 * gq] = ph[gq].x; h[4 * gq + 1] = ph[gq].y; h[4 * gq + 2] = ph[gq].z; h[4 * gq + 3] = ph[gq].w; }
                    vprev = pv;
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
            if (J > 0) ESme[c * CH + lane] = eout_s[lane];
            __syncwarp();                                      // orders every lane's ES store before lane 0's release
            if (lane == 0) st_release(p.prog_b + item, (unsigned)(C - c));
        }
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
    }
}

// ------------------------------------------------------------------------------------------------------------------
// small kernels: per-pair values from the item partials, objective, reduction over pairs, descent step
__global__ void finalize_values_kernel(const double* __restrict__ VP, const PairMeta* __restrict__ pm, int N, int NS,
                                       double inv_kappa, float* __restrict__ out_values, float* __restrict__ out_objective) {
    __shared__ double red[256];
    double local = 0.0;
    for (int ps = threadIdx.x; ps < N; ps += blockDim.x) {
        double s = 0.0;
        for (int J = 0; J < NS; ++J) s += VP[(long long)ps * NS + J];
        s *= inv_kappa;
        if (out_values) out_values[pm[ps].k] = (float)s;
        local += s;
    }
    // objective: fixed-shape tree over the block (deterministic)
    red[threadIdx.x] = local;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0 && out_objective) *out_objective = (float)red[0];
}

// G[e] = sum over pairs (schedule order, fp64 accumulator: deterministic, no atomics); optional descent step
__global__ void reduce_pairs_kernel(const float* __restrict__ Gk, int N, long long md, float* __restrict__ out_grad,
                                    float* __restrict__ Z, float step) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= md) return;
    double acc = 0.0;
    for (int ps = 0; ps < N; ++ps) acc += (double)Gk[(long long)ps * md + e];
    const float gsum = (float)acc;
    if (out_grad) out_grad[e] = gsum;
    if (Z) Z[e] = Z[e] - step * gsum;
}

__global__ void gd_update_kernel(float* __restrict__ Z, const float* __restrict__ G, long long count, float step) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < count) Z[e] = Z[e] - step * G[e];
}

}  // namespace sdtw
