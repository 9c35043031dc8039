// line.cuh -- the small-grid step kernel ("a persistent kernel for tiny grids"; S7 H6).
//
// For grids with at most 32 * U unknowns per line in both directions (U = 4 or 8: up to 128^2 / 256^2) the whole
// step loop of Algorithm 1 runs in ONE launch of ONE thread-block cluster: all `nsteps` time
// steps, two half-steps each, with a hardware cluster barrier (release / acquire) between half-steps instead of a
// kernel boundary.  The three fields (at most 1.5 MB) stay in L2 for the whole run.
//
// A grid line is solved whole, on chip, by one warp (the north_star's "line staged whole ... cyclic reduction /
// PCR with warp shuffles", PAPER.md:120-134 CRM_forward / cr_div / CRM_backward): lane l owns the U consecutive
// points p in [U l, U l + U).  With the half-step's own LU pivots from the host table (cp_p, inv_p for every p < n:
// exact, no stationarity assumption, KMAX >= 32 * 8) both elimination sweeps are first-order linear recurrences
//
//      y_p = cp_p y_{p-1} + inv_p r_p            x_p = y_p + cp_p x_{p+1}
//
// so the lane solves its unit from a zero carry, and the carries are the inclusive scan of the pairs
// (A_l, L_l) -> (A_l A_{l-1}, L_l + A_l L_{l-1}) over the 32 lanes: five shuffle rounds (Kogge-Stone), the
// scalar-coefficient equivalent of the log2(n+1) - 1 reduction levels of P:124-128.  Nothing is truncated: the result
// is the LU solution to rounding for ANY tau / h (the exact path for short lines, SURVEY.md 8c pin 7's edge case).
//
// x half-step: warp = grid row, a lane's points are 16-byte vectors of the row (coalesced).
// y half-step: a CTA takes a strip of 16 adjacent grid columns, brings it in with coalesced 16-byte loads,
//              transposes it through shared memory (strip[column][row]), then warp = column; results go back the same way.
#pragma once
#include "kernels.cuh"

namespace w2d {

struct LineArgs {
    const double* table;   // ROW_DOUBLES per half-step (or per period)
    int table_period;
    int* d_k;              // device: completed solves; read at the start, advanced by nsteps at the end
    int nsteps;            // time steps to run in this launch
    int ring;              // 3 or 4 buffers, roles by roles_of()
    int one_y;             // 1: scheme 1, the y half-step's right-hand side is the "cur" field itself
    void* bufs[4];
    int n1, n2;            // unknowns per x line / y line
    long long pitch;       // elements
    const void* src[2];    // compact source window per direction: [p - sp0][line - sl0] (line fastest), or NULL
    int win_i0, win_j0, win_w, win_h;
    double g2;             // 2 gamma
};

__device__ __forceinline__ void cluster_barrier()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ unsigned cluster_ctarank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned cluster_nctarank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
    return r;
}

// 16-byte global accesses that bypass L1 (the data of the previous half-step was written by other SMs)
template <typename T>
__device__ __forceinline__ void ldcg16(const T* p, T* v)
{
    if constexpr (sizeof(T) == 8) {
        const double2 t = __ldcg(reinterpret_cast<const double2*>(p));
        v[0] = t.x; v[1] = t.y;
    } else {
        const float4 t = __ldcg(reinterpret_cast<const float4*>(p));
        v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
    }
}
template <typename T>
__device__ __forceinline__ void st16(T* p, const T* v)
{
    if constexpr (sizeof(T) == 8) *reinterpret_cast<double2*>(p) = make_double2(v[0], v[1]);
    else *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
}

// One line, whole, in a warp.  wp/wc: this lane's U points of w_{n-1} / w_n (0 beyond the line); s: q * source values
// (or 0).  Returns x in wc.  p0 = U * lane; cp/iv: the half-step's pivots for p0 .. p0 + U - 1 (0 beyond the line).
template <typename T, int U>
__device__ __forceinline__ void solve_line_warp(T (&wp)[U], T (&wc)[U], const T (&qs)[U], const T (&cp)[U],
                                                const T (&iv)[U], T am, T c1, T g2, bool one, int lane)
{
    constexpr unsigned FULL = 0xffffffffu;
    T y[U];
    if (one) {
#pragma unroll
        for (int e = 0; e < U; ++e) y[e] = wc[e];                           // r = V (scheme 1's y half-step)
    } else {
        T wl = __shfl_up_sync(FULL, wp[U - 1], 1), wr = __shfl_down_sync(FULL, wp[0], 1);
        if (lane == 0) wl = T(0);                                            // (2.10): zero ghost values
        if (lane == 31) wr = T(0);
#pragma unroll
        for (int e = 0; e < U; ++e) {                                        // A1 / A3: right-hand side of (2.11) / (2.12)
            const T left = e == 0 ? wl : wp[e - 1], right = e == U - 1 ? wr : wp[e + 1];
            y[e] = fmaT(g2, wc[e], fmaT(am, left + right, fmaT(c1, wp[e], qs[e])));
        }
    }
    // forward elimination from a zero carry, A = product of the unit's cp
    T A = T(1), f = T(0);
#pragma unroll
    for (int e = 0; e < U; ++e) {
        f = fmaT(cp[e], f, y[e] * iv[e]);
        y[e] = f;
        A *= cp[e];
    }
    // inclusive scan: v = y at the end of this lane's unit with the true carry
    T a = A, v = f;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const T a2 = __shfl_up_sync(FULL, a, d), v2 = __shfl_up_sync(FULL, v, d);
        if (lane >= d) {
            v = fmaT(a, v2, v);
            a *= a2;
        }
    }
    T c = __shfl_up_sync(FULL, v, 1);                                        // y at the end of the previous unit
    if (lane == 0) c = T(0);
#pragma unroll
    for (int e = 0; e < U; ++e) {
        c *= cp[e];
        y[e] += c;
    }
    // back substitution from a zero carry: x_p = y_p + cp_p x_{p+1}
#pragma unroll
    for (int e = U - 2; e >= 0; --e) y[e] = fmaT(cp[e], y[e + 1], y[e]);
    a = A;
    v = y[0];
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const T a2 = __shfl_down_sync(FULL, a, d), v2 = __shfl_down_sync(FULL, v, d);
        if (lane + d < 32) {
            v = fmaT(a, v2, v);
            a *= a2;
        }
    }
    c = __shfl_down_sync(FULL, v, 1);                                        // x at the start of the next unit
    if (lane == 31) c = T(0);
#pragma unroll
    for (int e = U - 1; e >= 0; --e) {
        c *= cp[e];
        wc[e] = y[e] + c;
    }
}

// grid = one cluster of C CTAs; block = 32 * W threads.  Dynamic shared memory: two strips [16][RP] of T.
template <typename T, int U, int W>
__global__ void __launch_bounds__(32 * W, 1) wave2d_line_steps(const __grid_constant__ LineArgs a)
{
    constexpr int V = 16 / (int)sizeof(T);       // elements per 16 bytes
    constexpr int NV = U / V;                    // 16-byte vectors per lane
    constexpr int SC = 16;                       // columns per strip of the y half-step
    constexpr int KC = SC / V;                   // 16-byte chunks per strip row
    constexpr int RP = 32 * U + 1;               // strip row pitch (odd: the transposing stores spread over the banks)
    static_assert(U % V == 0 && 32 * U <= KMAX, "a lane owns whole 16-byte vectors; every pivot is tabulated");
    extern __shared__ __align__(16) unsigned char line_smem[];
    T* const s_prev = reinterpret_cast<T*>(line_smem);
    T* const s_cur = s_prev + SC * RP;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int cta = (int)cluster_ctarank(), ncta = (int)cluster_nctarank();
    const int k0 = *a.d_k;
    const int p0 = U * lane;
    const T g2 = static_cast<T>(a.g2);

    for (int hs = 0; hs < 2 * a.nsteps; ++hs) {
        const int nh = 2 * k0 + hs;
        const int d = nh & 1;
        const double* row = a.table + static_cast<size_t>(a.table_period ? nh % a.table_period : nh) * ROW_DOUBLES;
        const Roles R = roles_of(nh, a.ring);
        const T* const prev = static_cast<const T*>(a.bufs[R.prev]);
        const T* const cur = static_cast<const T*>(a.bufs[R.cur]);
        T* const out = static_cast<T*>(a.bufs[R.out]);
        const int n = d == 0 ? a.n1 : a.n2, nlines = d == 0 ? a.n2 : a.n1;
        const T am = static_cast<T>(row[ROW_AM]), q = static_cast<T>(row[ROW_Q]), c1 = static_cast<T>(row[ROW_C1]);
        const bool one = d == 1 && a.one_y != 0;
        T cp[U], iv[U];
#pragma unroll
        for (int e = 0; e < U; ++e) {            // beyond the line: cp = inv = 0 decouples the padding (x = 0 there)
            const bool in = p0 + e < n;
            cp[e] = in ? static_cast<T>(__ldg(row + ROW_CP + p0 + e)) : T(0);
            iv[e] = in ? static_cast<T>(__ldg(row + ROW_INVP + p0 + e)) : T(0);
        }
        const T* const src = static_cast<const T*>(a.src[d]);
        const int sl0 = d == 0 ? a.win_j0 : a.win_i0, snl = d == 0 ? a.win_h : a.win_w;
        const int sp0 = d == 0 ? a.win_i0 : a.win_j0, snp = d == 0 ? a.win_w : a.win_h;
        auto source = [&](int line, T (&qs)[U]) {
#pragma unroll
            for (int e = 0; e < U; ++e) qs[e] = T(0);
            if (src != nullptr && !one && line >= sl0 && line < sl0 + snl && p0 < sp0 + snp && p0 + U > sp0) {
#pragma unroll
                for (int e = 0; e < U; ++e) {
                    const int ps = p0 + e - sp0;
                    if (ps >= 0 && ps < snp) qs[e] = q * src[static_cast<size_t>(ps) * snl + (line - sl0)];
                }
            }
        };

        if (d == 0) {
            // ---- x half-step: one warp per grid row, lanes along the row
            const bool inrow = p0 < a.pitch;     // (pitch is a multiple of 16 elements >= U: a lane is in or out as a whole)
            for (int j = cta * W + warp; j < nlines; j += ncta * W) {
                T wp[U], wc[U], qs[U];
#pragma unroll
                for (int e = 0; e < U; ++e) wp[e] = wc[e] = T(0);
                const long long o = static_cast<long long>(j) * a.pitch + p0;
                if (inrow) {                     // pad columns beyond n1 are zero and stay zero
#pragma unroll
                    for (int c = 0; c < NV; ++c) {
                        if (!one) ldcg16(prev + o + c * V, wp + c * V);
                        ldcg16(cur + o + c * V, wc + c * V);
                    }
                }
                source(j, qs);
                solve_line_warp<T, U>(wp, wc, qs, cp, iv, am, c1, g2, one, lane);
                if (inrow) {
#pragma unroll
                    for (int c = 0; c < NV; ++c) st16(out + o + c * V, wc + c * V);
                }
            }
        } else {
            // ---- y half-step: strips of 16 grid columns per CTA, transposed through shared memory
            for (int c0 = SC * cta; c0 < nlines; c0 += SC * ncta) {
                const int kc = threadIdx.x % KC, r0 = threadIdx.x / KC;
                for (int r = r0; r < n; r += (32 * W) / KC) {
                    T vp[V], vc[V];
                    const long long o = static_cast<long long>(r) * a.pitch + c0 + kc * V;   // inside the pitch: c0 + 16 <= pitch
                    if (!one) ldcg16(prev + o, vp);
                    ldcg16(cur + o, vc);
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        if (!one) s_prev[(kc * V + e) * RP + r] = vp[e];
                        s_cur[(kc * V + e) * RP + r] = vc[e];
                    }
                }
                __syncthreads();
                for (int w = warp; w < SC; w += W) {            // warp = grid column c0 + w (pad columns solve zeros)
                    T wp[U], wc[U], qs[U];
#pragma unroll
                    for (int e = 0; e < U; ++e) {
                        const bool in = p0 + e < n;
                        wp[e] = in && !one ? s_prev[w * RP + p0 + e] : T(0);
                        wc[e] = in ? s_cur[w * RP + p0 + e] : T(0);
                    }
                    source(c0 + w, qs);
                    solve_line_warp<T, U>(wp, wc, qs, cp, iv, am, c1, g2, one, lane);
#pragma unroll
                    for (int e = 0; e < U; ++e)
                        if (p0 + e < n) s_cur[w * RP + p0 + e] = wc[e];   // only this warp ever touches column w
                }
                __syncthreads();
                for (int r = r0; r < n; r += (32 * W) / KC) {
                    T vo[V];
#pragma unroll
                    for (int e = 0; e < V; ++e) vo[e] = s_cur[(kc * V + e) * RP + r];
                    st16(out + static_cast<long long>(r) * a.pitch + c0 + kc * V, vo);
                }
                __syncthreads();                                  // the strips are reused by the next pass
            }
        }
        cluster_barrier();   // every store of this half-step is visible to every CTA of the cluster (release / acquire)
    }
    if (cta == 0 && threadIdx.x == 0) *a.d_k = k0 + a.nsteps;
}

}  // namespace w2d
