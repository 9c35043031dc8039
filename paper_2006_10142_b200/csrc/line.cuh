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

// ---- the same loop with the fields resident in the cluster's shared memory -----------------------------------------
// Between two half-steps the kernel above sends every field through L2 and separates the half-steps by a cluster barrier
// with release / acquire semantics -- which compiles to a GPU-wide memory barrier (MEMBAR.ALL.GPU ... CCTL.IVALL): about
// 3.5 us per half-step at 127^2, almost none of it arithmetic.  Here the time levels never leave the chip and no fence is
// executed in the loop.  CTA c of the cluster owns a block of grid rows and a block of grid columns and keeps
//      Xprev, Xcur[2] : w_{n-1}, w_n of its rows       (read by the x half-step)
//      Yprev, Ycur[2] : w_{n-1}, w_n of its columns    (read by the y half-step)
// in shared memory.  A level w_m is produced by a half-step of direction D and read twice: as "cur" by the next half-step
// (the other direction) and as "prev" by the one after (direction D again).  So the warp that solves a line overwrites the
// line's "prev" copy in place (its own CTA, same layout) and sends the values into the "cur" buffer of the CTAs that own
// the crossing lines: asynchronous distributed-shared-memory stores (st.async ... mbarrier::complete_tx::bytes) that
// count their bytes on an mbarrier of the RECEIVING CTA.  The receiver knows how many bytes a half-step sends it (its
// lines x their length) and waits for exactly that: a point-to-point hand-over, no cluster-wide barrier, no memory fence.
// The "cur" buffers are double-buffered by step parity: a CTA can run at most one half-step ahead of the slowest one
// (its next half-step needs everybody's contribution), so a buffer is never overwritten while it is still read.
// Global memory is touched at the start (load w_{n-1}, w_n) and at the end (store them) of a launch.
// A line is stored lane-interleaved: point p = U l + e sits at e * 32 + l, so lane l reads its U points conflict-free;
// lines are LP = 32 U + 1 apart, so the scatter (32 lanes, 32 different lines, one position) is conflict-free too.
// Scheme 0 only (the host keeps the kernel above for scheme 1 and for grids whose six buffers do not fit).
__device__ __forceinline__ uint32_t cluster_map(uint32_t local_smem_addr, unsigned cta)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_smem_addr), "r"(cta));
    return r;
}
// remote store that adds its size to the transaction count of the mbarrier `bar` (both addresses in the receiving CTA)
__device__ __forceinline__ void st_async(uint32_t addr, double v, uint32_t bar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];" ::"r"(addr),
                 "l"(__double_as_longlong(v)), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void st_async(uint32_t addr, float v, uint32_t bar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];" ::"r"(addr),
                 "r"(__float_as_uint(v)), "r"(bar)
                 : "memory");
}
// wait for the phase of parity `parity`; acquire at cluster scope: the bytes counted came from other CTAs
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "W2D_CWAIT:\n"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n"
        "@p bra W2D_CDONE;\n"
        "bra W2D_CWAIT;\n"
        "W2D_CDONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}

template <typename T, int U, int W>
__global__ void __launch_bounds__(32 * W, 1) wave2d_line_resident(const __grid_constant__ LineArgs a)
{
    constexpr int V = 16 / (int)sizeof(T), NV = U / V;
    constexpr int LP = 32 * U + 1;               // elements between the lines of a buffer
    static_assert(U % V == 0 && 32 * U <= KMAX, "a lane owns whole 16-byte vectors; every pivot is tabulated");
    extern __shared__ __align__(16) unsigned char line_smem[];
    __shared__ __align__(8) unsigned long long s_bar[2][2];   // [direction of the receiving half-step][step parity]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int cta = (int)cluster_ctarank(), ncta = (int)cluster_nctarank();
    const int rpc = (a.n2 + ncta - 1) / ncta, cpc = (a.n1 + ncta - 1) / ncta;    // rows / columns per CTA
    const int lb = rpc > cpc ? rpc : cpc;                                       // lines per buffer
    T* const Xprev = reinterpret_cast<T*>(line_smem);
    T* const Yprev = Xprev + lb * LP;
    T* const Xcur = Yprev + lb * LP;             // [2][lb][LP]
    T* const Ycur = Xcur + 2 * lb * LP;          // [2][lb][LP]
    const int j0 = cta * rpc, i0 = cta * cpc;
    const int nrows = min(rpc, max(a.n2 - j0, 0)), ncols = min(cpc, max(a.n1 - i0, 0));   // lines this CTA owns
    // bytes a half-step sends this CTA: every line of the other direction, its values on the lines owned here
    const uint32_t bytes_x = static_cast<uint32_t>(a.n1) * nrows * (uint32_t)sizeof(T);    // into Xcur (by a y half-step)
    const uint32_t bytes_y = static_cast<uint32_t>(a.n2) * ncols * (uint32_t)sizeof(T);    // into Ycur (by an x half-step)
    const int k0 = *a.d_k;
    const int p0 = U * lane;
    const T g2 = static_cast<T>(a.g2);
    auto pos = [](int p) { return (p % U) * 32 + p / U; };   // place of point p inside a stored line

    // ---- start: zero the buffers (points beyond a line stay 0), then w_{n-1}, w_n of this CTA's rows and w_n of its columns
    for (int i = threadIdx.x; i < 6 * lb * LP; i += 32 * W) Xprev[i] = T(0);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int b = 0; b < 4; ++b) mbar_init(smem_u32(&s_bar[b >> 1][b & 1]), 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (threadIdx.x == 0) {      // first use of every barrier (Xcur[0] is first filled from global memory below: its barrier
                                 // waits for the y half-step of step 1)
        mbar_arrive_expect_tx(smem_u32(&s_bar[0][0]), bytes_x);
        mbar_arrive_expect_tx(smem_u32(&s_bar[0][1]), bytes_x);
        mbar_arrive_expect_tx(smem_u32(&s_bar[1][0]), bytes_y);
        mbar_arrive_expect_tx(smem_u32(&s_bar[1][1]), bytes_y);
    }
    {
        const Roles R = roles_of(2 * k0, a.ring);
        const T* const prev = static_cast<const T*>(a.bufs[R.prev]);
        const T* const cur = static_cast<const T*>(a.bufs[R.cur]);
        for (int lj = warp; lj < nrows; lj += W) {
            if (p0 < a.pitch) {
                T wp[U], wc[U];
                const long long o = static_cast<long long>(j0 + lj) * a.pitch + p0;
#pragma unroll
                for (int c = 0; c < NV; ++c) {
                    ldcg16(prev + o + c * V, wp + c * V);
                    ldcg16(cur + o + c * V, wc + c * V);
                }
#pragma unroll
                for (int e = 0; e < U; ++e) {
                    Xprev[lj * LP + e * 32 + lane] = wp[e];
                    Xcur[lj * LP + e * 32 + lane] = wc[e];
                }
            }
        }
        for (int idx = threadIdx.x; idx < a.n2 * cpc; idx += 32 * W) {   // columns: cpc consecutive values of every row
            const int j = idx / cpc, lc = idx - j * cpc;
            if (lc < ncols) Yprev[lc * LP + pos(j)] = __ldcg(cur + static_cast<long long>(j) * a.pitch + i0 + lc);
        }
    }
    // where this lane's U results of a line go: the "cur" buffer (parity 0) of the CTA that owns the crossing line, and that
    // CTA's barriers
    uint32_t to_y[U], to_x[U], bar_y[U], bar_x[U];
#pragma unroll
    for (int e = 0; e < U; ++e) {
        const int i = min(p0 + e, a.n1 - 1), j = min(p0 + e, a.n2 - 1);
        to_y[e] = cluster_map(smem_u32(Ycur + (i % cpc) * LP), static_cast<unsigned>(i / cpc));
        to_x[e] = cluster_map(smem_u32(Xcur + (j % rpc) * LP), static_cast<unsigned>(j / rpc));
        bar_y[e] = cluster_map(smem_u32(&s_bar[1][0]), static_cast<unsigned>(i / cpc));
        bar_x[e] = cluster_map(smem_u32(&s_bar[0][0]), static_cast<unsigned>(j / rpc));
    }
    const uint32_t half = static_cast<uint32_t>(lb * LP * (int)sizeof(T));   // bytes between the two parities of a buffer
    // pivots of both directions stay in registers when the table has period 2 (constant c and g)
    T cpx[U], ivx[U], cpy[U], ivy[U];
    auto load_pivots = [&](const double* row, T (&cp)[U], T (&iv)[U], int n) {
#pragma unroll
        for (int e = 0; e < U; ++e) {            // beyond the line: cp = inv = 0 decouples the padding (x = 0 there)
            const bool in = p0 + e < n;
            cp[e] = in ? static_cast<T>(__ldg(row + ROW_CP + p0 + e)) : T(0);
            iv[e] = in ? static_cast<T>(__ldg(row + ROW_INVP + p0 + e)) : T(0);
        }
    };
    const bool periodic = a.table_period == 2;
    if (periodic) {
        load_pivots(a.table, cpx, ivx, a.n1);
        load_pivots(a.table + ROW_DOUBLES, cpy, ivy, a.n2);
    }
    cluster_barrier();             // every CTA's buffers and barriers are initialised before anybody sends to them

    for (int hs = 0; hs < 2 * a.nsteps; ++hs) {
        const int t = hs >> 1, d = hs & 1;       // (a launch starts with an x half-step: nh = 2 k0 + hs)
        const int nh = 2 * k0 + hs;
        const double* row = a.table + static_cast<size_t>(a.table_period ? nh % a.table_period : nh) * ROW_DOUBLES;
        const int n = d == 0 ? a.n1 : a.n2;
        const T am = static_cast<T>(__ldg(row + ROW_AM)), q = static_cast<T>(__ldg(row + ROW_Q)), c1 = static_cast<T>(__ldg(row + ROW_C1));
        T cp[U], iv[U];
        if (!periodic) {
            load_pivots(row, cp, iv, n);
        } else {
#pragma unroll
            for (int e = 0; e < U; ++e) {
                cp[e] = d == 0 ? cpx[e] : cpy[e];
                iv[e] = d == 0 ? ivx[e] : ivy[e];
            }
        }
        const T* const src = static_cast<const T*>(a.src[d]);
        const int sl0 = d == 0 ? a.win_j0 : a.win_i0, snl = d == 0 ? a.win_h : a.win_w;
        const int sp0 = d == 0 ? a.win_i0 : a.win_j0, snp = d == 0 ? a.win_w : a.win_h;
        // x half-step of step t reads Xcur[t & 1] (filled by the y half-step of step t - 1) and sends into Ycur[t & 1];
        // y half-step of step t reads Ycur[t & 1] and sends into Xcur[(t + 1) & 1]
        const int rb = t & 1, sb = d == 0 ? (t & 1) : ((t + 1) & 1);
        T* const bprev = d == 0 ? Xprev : Yprev;
        const T* const bcur = (d == 0 ? Xcur : Ycur) + rb * lb * LP;
        if (!(d == 0 && t == 0)) {               // wait for this half-step's input: every byte the previous one sent here
            const uint32_t bar = smem_u32(&s_bar[d][rb]);
            const int use = d == 0 ? (t - 1) >> 1 : t >> 1;        // how often this barrier has completed before
            mbar_wait_cluster(bar, use & 1);
            __syncthreads();                     // (nobody still polls the phase that is re-armed now)
            if (threadIdx.x == 0) mbar_arrive_expect_tx(bar, d == 0 ? bytes_x : bytes_y);   // its next use, two steps on
        }
        const int nl = d == 0 ? nrows : ncols, l0 = d == 0 ? j0 : i0;
        for (int ll = warp; ll < nl; ll += W) {
            const int line = l0 + ll;
            T wp[U], wc[U], qs[U];
#pragma unroll
            for (int e = 0; e < U; ++e) {
                wp[e] = bprev[ll * LP + e * 32 + lane];
                wc[e] = bcur[ll * LP + e * 32 + lane];
                qs[e] = T(0);
            }
            if (src != nullptr && line >= sl0 && line < sl0 + snl && p0 < sp0 + snp && p0 + U > sp0) {
#pragma unroll
                for (int e = 0; e < U; ++e) {
                    const int ps = p0 + e - sp0;
                    if (ps >= 0 && ps < snp) qs[e] = q * src[static_cast<size_t>(ps) * snl + (line - sl0)];
                }
            }
            solve_line_warp<T, U>(wp, wc, qs, cp, iv, am, c1, g2, false, lane);
            const uint32_t off = static_cast<uint32_t>(pos(line) * (int)sizeof(T)) + (sb ? half : 0u);
            const uint32_t boff = sb ? 8u : 0u;
#pragma unroll
            for (int e = 0; e < U; ++e) {
                bprev[ll * LP + e * 32 + lane] = wc[e];                       // "prev" of this direction's next half-step
                if (p0 + e < n) {                                              // "cur" of the other direction's
                    if (d == 0) st_async(to_y[e] + off, wc[e], bar_y[e] + boff);
                    else st_async(to_x[e] + off, wc[e], bar_x[e] + boff);
                }
            }
        }
    }

    // ---- end: w_{n-1}, w_n of this CTA's rows go back to the ring in global memory
    {
        const int t = a.nsteps, rb = t & 1;      // Xcur[t & 1] is what an x half-step of step t would read
        if (t > 0) mbar_wait_cluster(smem_u32(&s_bar[0][rb]), ((t - 1) >> 1) & 1);
        const Roles R = roles_of(2 * (k0 + a.nsteps), a.ring);
        T* const prev = static_cast<T*>(a.bufs[R.prev]);
        T* const cur = static_cast<T*>(a.bufs[R.cur]);
        const T* const xc = Xcur + rb * lb * LP;
        for (int lj = warp; lj < nrows; lj += W) {
            if (p0 < a.pitch) {
                T wp[U], wc[U];
#pragma unroll
                for (int e = 0; e < U; ++e) {
                    wp[e] = Xprev[lj * LP + e * 32 + lane];
                    wc[e] = xc[lj * LP + e * 32 + lane];
                }
                const long long o = static_cast<long long>(j0 + lj) * a.pitch + p0;
#pragma unroll
                for (int c = 0; c < NV; ++c) {
                    st16(prev + o + c * V, wp + c * V);
                    st16(cur + o + c * V, wc + c * V);
                }
            }
        }
    }
    if (cta == 0 && threadIdx.x == 0) *a.d_k = k0 + a.nsteps;
    cluster_barrier();   // no CTA leaves while another may still send to it
}

}  // namespace w2d
