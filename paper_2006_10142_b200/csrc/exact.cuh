// exact.cuh -- the untruncated line solvers (solver EXACT): any tau / h, any line length up to 16384 unknowns.
//
// The north_star's solver sketch -- a line "staged whole in shared memory ... solved by cyclic reduction (or PCR
// for the last levels) with warp shuffles" (CRM_forward, cr_div, CRM_backward) -- with the two
// changes the scalar coefficients allow:
//   * register blocking: a thread owns U = 8 consecutive points and eliminates them serially (the first log2 U
//     reduction levels happen in registers, no strided shared-memory access, no bank conflicts);
//   * the remaining levels are a scan: with the LU pivots cp_p, inv_p of the half-step's Toeplitz matrix both sweeps
//     are first-order linear recurrences, so the carries between units follow from the inclusive scan of the pairs
//     (A, L) -> (A A', L + A L') -- five shuffle rounds inside a warp, one more scan over the warp aggregates of the
//     line in shared memory.  That is the log2(n+1) - 1 levels of P:124-128 with 2 CTA barriers per sweep direction.
// Nothing is truncated, so the result is the LU solution to rounding for every tau / h.
//
// x half-step (lines = grid rows): a group of warps owns a row; a thread's points are 16-byte vectors of the row
//   (coalesced, straight into registers).  Lines longer than one pass of the CTA (n > 4096) are walked in segments:
//   forward left to right with the carry, y parked in shared memory (a 16384-point fp64 line is 128 KB), then
//   backward right to left.
// y half-step (lines = grid columns): a CTA takes a strip of SC adjacent columns over ALL rows; coalesced 16-byte
//   loads assemble the right-hand side (A3) straight into a shared-memory strip [column][row] (the only staging: one
//   value per point), the columns are solved in place by the same block-wide scan, and the strip is written back
//   with coalesced stores.  SC is the widest strip that fits 200 KB (4 columns at n2 = 4095 in fp64).  No transpose
//   pass, no second trip through HBM: each sweep reads 2 fields and writes 1.
#pragma once
#include "kernels.cuh"

namespace w2d {

constexpr int EX_U = 8;          // points per thread
constexpr int EX_NT = 512;       // threads per CTA
constexpr int EX_NW = EX_NT / 32;

// cpv[p], ivv[p], p < n: the LU pivots of tridiag(-ap, beta, -ap).  The first KMAX come from the host table; if the
// recurrence has not reached its fixed point (rho, 1 / (beta - ap rho)) by then, one thread continues it until it has
// (to 1e-15 relative), and the rest is filled in parallel.  conv[0] = first index from which every pivot is the fixed
// point to 2e-15: units beyond it take the stationary fast path of the solvers.
__global__ void wave2d_exact_pivots(const double* table, int period, const int* d_k, int n_off, int n, double* cpv,
                                    double* ivv, int* conv)
{
    __shared__ int s_conv, s_head;
    const int nh = n_off + 2 * (*d_k);
    const double* row = table + static_cast<size_t>(period ? nh % period : nh) * ROW_DOUBLES;
    const double ap = row[ROW_AP], beta = row[ROW_BETA], rho = row[ROW_RHO], inv = row[ROW_INV];
    const int head = n < KMAX ? n : KMAX;
    if (threadIdx.x == 0) s_head = 0;
    __syncthreads();
    for (int p = threadIdx.x; p < head; p += blockDim.x) {
        const double c = row[ROW_CP + p], v = row[ROW_INVP + p];
        cpv[p] = c;
        ivv[p] = v;
        if (!(fabs(c - rho) <= 2e-15 * rho && fabs(v - inv) <= 2e-15 * inv)) atomicMax(&s_head, p + 1);
    }
    __syncthreads();
    if (n <= KMAX || s_head < KMAX) {           // stationary inside the table: the rest is the fixed point
        for (int p = KMAX + threadIdx.x; p < n; p += blockDim.x) {
            cpv[p] = rho;
            ivv[p] = inv;
        }
        if (threadIdx.x == 0) conv[0] = s_head;
        return;
    }
    if (threadIdx.x == 0) {
        double cp = cpv[KMAX - 1];
        int p = KMAX;
        for (; p < n; ++p) {
            const double iv = 1.0 / (beta - ap * cp);
            cp = ap * iv;
            cpv[p] = cp;
            ivv[p] = iv;
            if (fabs(cp - rho) <= 1e-15 * rho && fabs(iv - inv) <= 1e-15 * inv) { ++p; break; }
        }
        s_conv = p;
        conv[0] = p;
    }
    __syncthreads();
    for (int p = s_conv + threadIdx.x; p < n; p += blockDim.x) {
        cpv[p] = rho;
        ivv[p] = inv;
    }
}

// Stationary scalars of a half-step (units whose pivots are all the fixed point): rho^(e+1), A = rho^U and its powers.
template <typename T, int U>
struct Stat {
    T rho, inv;
    T pw[U];      // rho^(e+1)
    T Ap[6];      // A^(2^d), d = 0..5 (A^32 = a whole warp)
    T Alane;      // A^lane
    T Arev;       // A^(31 - lane)
    __device__ __forceinline__ void init(double rho_d, double inv_d, int lane)
    {
        rho = static_cast<T>(rho_d);
        inv = static_cast<T>(inv_d);
        double pwr = rho_d;
#pragma unroll
        for (int e = 0; e < U; ++e, pwr *= rho_d) pw[e] = static_cast<T>(pwr);
        double A = pw[U - 1];
#pragma unroll
        for (int d = 0; d < 6; ++d, A *= A) Ap[d] = static_cast<T>(A);
        Alane = static_cast<T>(pow(static_cast<double>(pw[U - 1]), static_cast<double>(lane)));
        Arev = static_cast<T>(pow(static_cast<double>(pw[U - 1]), static_cast<double>(31 - lane)));
    }
};

// ---- block-wide solve of one line segment ------------------------------------------------------------------
// A "group" is wpc consecutive warps of the CTA; thread (gw, lane) of the group owns unit gw * 32 + lane of the segment.
// sA, sL (forward) and sB, sH (backward) are the group's slices [wpc] of the CTA's aggregate arrays.  Every thread of
// the CTA must call these (they contain one CTA barrier each).

// y[] holds r on entry and the true y on exit.  cin: y just before the segment.  Returns y at the end of the segment.
// FAST (warp-uniform): all 32 units of this warp are whole and stationary -- cp = rho, inv constant, A = rho^U, so the
// scan needs no products and half the shuffles; cp[] / iv[] are not read.
template <typename T, int U, bool FAST>
__device__ __forceinline__ T group_forward_impl(T (&y)[U], const T (&cp)[U], const T (&iv)[U], const Stat<T, U>& S,
                                                T cin, int wpc, int gw, int lane, T* sA, T* sL)
{
    constexpr unsigned FULL = 0xffffffffu;
    T a, v;
    if constexpr (FAST) {
        T f = y[0] * S.inv;
        y[0] = f;
#pragma unroll
        for (int e = 1; e < U; ++e) {
            f = fmaT(S.rho, f, y[e] * S.inv);
            y[e] = f;
        }
        v = f;
#pragma unroll
        for (int d = 0; d < 5; ++d) {
            const T v2 = __shfl_up_sync(FULL, v, 1 << d);
            if (lane >= (1 << d)) v = fmaT(S.Ap[d], v2, v);
        }
        a = S.Ap[5];                                   // (lane 31's prefix product: the whole warp)
    } else {
        T A = T(1), f = T(0);
#pragma unroll
        for (int e = 0; e < U; ++e) {
            f = fmaT(cp[e], f, y[e] * iv[e]);
            y[e] = f;
            A *= cp[e];
        }
        a = A;
        v = f;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const T a2 = __shfl_up_sync(FULL, a, d), v2 = __shfl_up_sync(FULL, v, d);
            if (lane >= d) {
                v = fmaT(a, v2, v);
                a *= a2;
            }
        }
    }
    if (lane == 31) {
        sA[gw] = a;
        sL[gw] = v;
    }
    named_bar_sync(1, EX_NT);   // (fast and general warps arrive from different copies of this code)
    T ga = lane < wpc ? sA[lane] : T(1), gv = lane < wpc ? sL[lane] : T(0);
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const T a2 = __shfl_up_sync(FULL, ga, d), v2 = __shfl_up_sync(FULL, gv, d);
        if (lane >= d) {
            gv = fmaT(ga, v2, gv);
            ga *= a2;
        }
    }
    const int gp = gw > 0 ? gw - 1 : 0;
    T cw = fmaT(__shfl_sync(FULL, ga, gp), cin, __shfl_sync(FULL, gv, gp));   // y entering this warp
    if (gw == 0) cw = cin;
    const T cout = fmaT(__shfl_sync(FULL, ga, wpc - 1), cin, __shfl_sync(FULL, gv, wpc - 1));
    const T pv = __shfl_up_sync(FULL, v, 1);
    if constexpr (FAST) {
        const T c = lane == 0 ? cw : fmaT(S.Alane, cw, pv);   // y at the end of the previous unit
#pragma unroll
        for (int e = 0; e < U; ++e) y[e] = fmaT(S.pw[e], c, y[e]);
    } else {
        const T pa = __shfl_up_sync(FULL, a, 1);
        T c = lane == 0 ? cw : fmaT(pa, cw, pv);
#pragma unroll
        for (int e = 0; e < U; ++e) {
            c *= cp[e];
            y[e] += c;
        }
    }
    return cout;
}

// y[] holds the true y on entry and x on exit.  xin: x just after the segment.  Returns x at the start of the segment.
template <typename T, int U, bool FAST>
__device__ __forceinline__ T group_backward_impl(T (&y)[U], const T (&cp)[U], const Stat<T, U>& S, T xin, int wpc,
                                                 int gw, int lane, T* sB, T* sH)
{
    constexpr unsigned FULL = 0xffffffffu;
    T a, v;
    if constexpr (FAST) {
#pragma unroll
        for (int e = U - 2; e >= 0; --e) y[e] = fmaT(S.rho, y[e + 1], y[e]);
        v = y[0];
#pragma unroll
        for (int d = 0; d < 5; ++d) {
            const T v2 = __shfl_down_sync(FULL, v, 1 << d);
            if (lane + (1 << d) < 32) v = fmaT(S.Ap[d], v2, v);
        }
        a = S.Ap[5];
    } else {
        T A = cp[U - 1];
#pragma unroll
        for (int e = U - 2; e >= 0; --e) {
            y[e] = fmaT(cp[e], y[e + 1], y[e]);
            A *= cp[e];
        }
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
    }
    if (lane == 0) {
        sB[gw] = a;
        sH[gw] = v;
    }
    named_bar_sync(1, EX_NT);
    T ga = lane < wpc ? sB[lane] : T(1), gv = lane < wpc ? sH[lane] : T(0);
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const T a2 = __shfl_down_sync(FULL, ga, d), v2 = __shfl_down_sync(FULL, gv, d);
        if (lane + d < 32) {
            gv = fmaT(ga, v2, gv);
            ga *= a2;
        }
    }
    const int gn = gw + 1 < wpc ? gw + 1 : gw;
    T xw = fmaT(__shfl_sync(FULL, ga, gn), xin, __shfl_sync(FULL, gv, gn));   // x entering this warp from the right
    if (gw + 1 >= wpc) xw = xin;
    const T cout = fmaT(__shfl_sync(FULL, ga, 0), xin, __shfl_sync(FULL, gv, 0));
    const T nv = __shfl_down_sync(FULL, v, 1);
    if constexpr (FAST) {
        const T c = lane == 31 ? xw : fmaT(S.Arev, xw, nv);   // x at the start of the next unit
#pragma unroll
        for (int e = 0; e < U; ++e) y[e] = fmaT(S.pw[U - 1 - e], c, y[e]);
    } else {
        const T na = __shfl_down_sync(FULL, a, 1);
        T c = lane == 31 ? xw : fmaT(na, xw, nv);
#pragma unroll
        for (int e = U - 1; e >= 0; --e) {
            c *= cp[e];
            y[e] += c;
        }
    }
    return cout;
}

// fast: warp-uniform (see above).  Both variants hold exactly one CTA barrier, so warps of one CTA may differ.
template <typename T, int U>
__device__ __forceinline__ T group_forward(bool fast, T (&y)[U], const T (&cp)[U], const T (&iv)[U], const Stat<T, U>& S,
                                           T cin, int wpc, int gw, int lane, T* sA, T* sL)
{
    return fast ? group_forward_impl<T, U, true>(y, cp, iv, S, cin, wpc, gw, lane, sA, sL)
                : group_forward_impl<T, U, false>(y, cp, iv, S, cin, wpc, gw, lane, sA, sL);
}
template <typename T, int U>
__device__ __forceinline__ T group_backward(bool fast, T (&y)[U], const T (&cp)[U], const Stat<T, U>& S, T xin, int wpc,
                                            int gw, int lane, T* sB, T* sH)
{
    return fast ? group_backward_impl<T, U, true>(y, cp, S, xin, wpc, gw, lane, sB, sH)
                : group_backward_impl<T, U, false>(y, cp, S, xin, wpc, gw, lane, sB, sH);
}

// ---- variable speed: the pivots of a non-Toeplitz line -------------------------------------------
// With c(t) cs(x,y) the system of a line is  -a_p x_{p-1} + (gamma + 2 a_p) x_p - a_p x_{p+1} = r_p,  a_p = ap cs_p
// (Algorithm 1's a_i, b_i, c_i "per point"), and the elimination pivots follow the NONLINEAR recurrence
//      cp_p = a_p / (b_p - a_p cp_{p-1}),    inv_p = 1 / (b_p - a_p cp_{p-1}),      b_p = gamma + 2 a_p.
// It is a linear-fractional map of cp_{p-1}, so maps compose as 2x2 matrices: with cp = N / D,
//      (N, D) <- (a_p D, b_p D - a_p N).
// A thread multiplies the maps of its U points, the products are scanned over the line exactly like the carries
// (normalised to [[A, B], [C, 1]] after every product: the maps are projective, and C B' + 1 >= 3/4 by diagonal
// dominance), and the exclusive prefix applied to the value entering the segment gives every thread its cp_{p0-1}.
template <typename T>
struct Mob {
    T A, B, C;   // [[A, B], [C, 1]]
};
template <typename T>
__device__ __forceinline__ T rcpT(T x) { return T(1) / x; }
// `later` after `earlier`
template <typename T>
__device__ __forceinline__ Mob<T> mob_after(const Mob<T>& later, const Mob<T>& earlier)
{
    const T d = rcpT(fmaT(later.C, earlier.B, T(1)));
    Mob<T> r;
    r.A = fmaT(later.A, earlier.A, later.B * earlier.C) * d;
    r.B = fmaT(later.A, earlier.B, later.B) * d;
    r.C = fmaT(later.C, earlier.A, earlier.C) * d;
    return r;
}
template <typename T>
__device__ __forceinline__ T mob_apply(const Mob<T>& m, T c) { return fmaT(m.A, c, m.B) * rcpT(fmaT(m.C, c, T(1))); }

// a[]: this thread's a_p (0 beyond the line).  cin: cp just before the segment.  Fills cp[], iv[]; returns cp at the end
// of the segment.  sM: the group's slice [3][wpc] of a CTA array (one CTA barrier inside; every thread must call).
template <typename T, int U>
__device__ __forceinline__ T group_pivots(const T (&a)[U], T gamma, T (&cp)[U], T (&iv)[U], T cin, int wpc, int gw,
                                          int lane, T* sMA, T* sMB, T* sMC)
{
    constexpr unsigned FULL = 0xffffffffu;
    // the unit's map: rows (n0, n1), (d0, d1) of N and D as linear forms of the (N, D) entering the unit
    T n0 = T(1), n1 = T(0), d0 = T(0), d1 = T(1);
#pragma unroll
    for (int e = 0; e < U; ++e) {
        const T b = fmaT(T(2), a[e], gamma);
        const T m0 = a[e] * d0, m1 = a[e] * d1;
        d0 = fmaT(b, d0, -(a[e] * n0));
        d1 = fmaT(b, d1, -(a[e] * n1));
        n0 = m0;
        n1 = m1;
        if ((e & 3) == 3) {                      // keep the entries in range (fp32: b^8 may not fit)
            const T sc = rcpT(d1);
            n0 *= sc; n1 *= sc; d0 *= sc; d1 = T(1);
        }
    }
    Mob<T> m{n0, n1, d0};                        // (d1 == 1 after the last normalisation: U is a multiple of 4)
    static_assert(U % 4 == 0, "the unit map is normalised every 4 points");
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {           // inclusive scan over the lanes
        Mob<T> o;
        o.A = __shfl_up_sync(FULL, m.A, d);
        o.B = __shfl_up_sync(FULL, m.B, d);
        o.C = __shfl_up_sync(FULL, m.C, d);
        if (lane >= d) m = mob_after(m, o);
    }
    if (lane == 31) {
        sMA[gw] = m.A;
        sMB[gw] = m.B;
        sMC[gw] = m.C;
    }
    named_bar_sync(1, EX_NT);
    Mob<T> g;
    g.A = lane < wpc ? sMA[lane] : T(1);
    g.B = lane < wpc ? sMB[lane] : T(0);
    g.C = lane < wpc ? sMC[lane] : T(0);
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {           // inclusive scan over the warps of the group (identity beyond wpc)
        Mob<T> o;
        o.A = __shfl_up_sync(FULL, g.A, d);
        o.B = __shfl_up_sync(FULL, g.B, d);
        o.C = __shfl_up_sync(FULL, g.C, d);
        if (lane >= d) g = mob_after(g, o);
    }
    const int gp = gw > 0 ? gw - 1 : 0;
    Mob<T> pw;                                   // everything before this warp
    pw.A = __shfl_sync(FULL, g.A, gp);
    pw.B = __shfl_sync(FULL, g.B, gp);
    pw.C = __shfl_sync(FULL, g.C, gp);
    const T cw = gw == 0 ? cin : mob_apply(pw, cin);
    Mob<T> all;
    all.A = __shfl_sync(FULL, g.A, wpc - 1);
    all.B = __shfl_sync(FULL, g.B, wpc - 1);
    all.C = __shfl_sync(FULL, g.C, wpc - 1);
    const T cout = mob_apply(all, cin);
    Mob<T> pl;                                   // the lanes before this one
    pl.A = __shfl_up_sync(FULL, m.A, 1);
    pl.B = __shfl_up_sync(FULL, m.B, 1);
    pl.C = __shfl_up_sync(FULL, m.C, 1);
    T c = lane == 0 ? cw : mob_apply(pl, cw);    // cp_{p0 - 1}
#pragma unroll
    for (int e = 0; e < U; ++e) {
        const T b = fmaT(T(2), a[e], gamma);
        const T v = rcpT(fmaT(-a[e], c, b));
        c = a[e] * v;
        cp[e] = c;
        iv[e] = v;
    }
    return cout;
}

struct ExactArgs {
    FieldSet fs;
    const double* table;
    int period;
    const int* d_k;
    int n_off;
    int n, nlines;
    long long pitch;
    const double* cpv;     // pivots of this half-step (wave2d_exact_pivots)
    const double* ivv;
    const int* conv;       // first index from which the pivots are the fixed point
    const void* src;       // compact source window [p - sp0][line - sl0], or NULL
    int sl0, snl, sp0, snp;
    double g2;
    int one;               // scheme 1's y half-step: right-hand side = the "cur" field
    int wpc;               // warps per line (group size); EX_NW / wpc lines per CTA pass
    int nseg;              // x: segments of wpc * 32 * U points per line (nseg > 1 only with wpc == EX_NW)
    int sc;                // y: columns per strip
    const void* cs;        // VAR kernels: spatial speed factor (pitched like a field, pad 0)
    double gamma;          // VAR kernels: the time-quotient constant (b_p = gamma + 2 a_p)
};

template <typename T>
__device__ __forceinline__ void ld16(const T* p, T* v)
{
    if constexpr (sizeof(T) == 8) {
        const double2 t = *reinterpret_cast<const double2*>(p);
        v[0] = t.x; v[1] = t.y;
    } else {
        const float4 t = *reinterpret_cast<const float4*>(p);
        v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
    }
}
template <typename T>
__device__ __forceinline__ void st16g(T* p, const T* v)
{
    if constexpr (sizeof(T) == 8) *reinterpret_cast<double2*>(p) = make_double2(v[0], v[1]);
    else *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
}

// per-thread asynchronous copies global -> shared (LDGSTS): a thread prefetches its own points of the next row
__device__ __forceinline__ void cp_async16(void* dst, const void* src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
template <int BYTES>
__device__ __forceinline__ void cp_async_small(void* dst, const void* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(smem_u32(dst)), "l"(src), "n"(BYTES) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- x half-step: (A1 + A2) exact ------------------------------------------------------------------------------
// grid: CTAs loop over passes of EX_NW / wpc rows.  Dynamic shared memory:
//   nseg == 1: two prefetch slots of EX_NT * (2 NV + 1) 16-byte cells -- while a pass is solved, every thread's own
//              points of the next pass's row (and the two neighbour values of a warp) are already on their way;
//   nseg  > 1: the parked line, nseg * wpc * 32 * U values (no prefetch: the line itself fills shared memory).
// VAR: variable speed -- one more field (cs) per row, the pivots come from group_pivots, no stationary fast path.
template <typename T, bool VAR>
__global__ void __launch_bounds__(EX_NT) wave2d_exact_x(const __grid_constant__ ExactArgs a)
{
    constexpr int U = EX_U, V = 16 / (int)sizeof(T), NV = U / V;
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ __align__(16) unsigned char ex_smem[];
    T* const s_line = reinterpret_cast<T*>(ex_smem);
    // aggregates of the block-wide scans, double-buffered: consecutive forward (or backward) calls alternate, so a warp
    // that runs ahead into the next call never overwrites what a slower warp still reads (one barrier per call)
    __shared__ T s_agg[2][4][EX_NW];
    __shared__ T s_mob[VAR ? 2 : 1][3][EX_NW];   // aggregates of the pivot scan (VAR), double-buffered likewise

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wpc = a.wpc, group = warp / wpc, gw = warp % wpc, ngroups = EX_NW / wpc;
    const int nh = a.n_off + 2 * (*a.d_k);
    const Roles R = roles_of(nh, a.fs.ring);
    const T* const prev = static_cast<const T*>(a.fs.b[R.prev]);
    const T* const cur = static_cast<const T*>(a.fs.b[R.cur]);
    T* const out = static_cast<T*>(a.fs.b[R.out]);
    [[maybe_unused]] const T* const csf = static_cast<const T*>(a.cs);
    const double* row = a.table + static_cast<size_t>(a.period ? nh % a.period : nh) * ROW_DOUBLES;
    const T am = static_cast<T>(row[ROW_AM]), q = static_cast<T>(row[ROW_Q]), c1 = static_cast<T>(row[ROW_C1]);
    [[maybe_unused]] const T ap = static_cast<T>(row[ROW_AP]), gam = static_cast<T>(a.gamma);
    const T g2 = static_cast<T>(a.g2);
    const bool one = a.one != 0;
    const int n = a.n, seg_pts = wpc * 32 * U;
    const T* const src = static_cast<const T*>(a.src);
    int pf = 0, pb = 0;   // buffer parity of the next forward / backward call
    [[maybe_unused]] int pp = 0;

    auto pivots = [&](int p0, T (&cp)[U], T (&iv)[U]) {
#pragma unroll
        for (int e = 0; e < U; ++e) {            // beyond the line: cp = inv = 0 decouples the padding (x = 0 there)
            const bool in = p0 + e < n;
            cp[e] = in ? static_cast<T>(a.cpv[p0 + e]) : T(0);
            iv[e] = in ? static_cast<T>(a.ivv[p0 + e]) : T(0);
        }
    };
    Stat<T, U> S;
    S.init(row[ROW_RHO], row[ROW_INV], lane);
    const int pc = VAR ? 0x7fffffff : *a.conv;    // pivots are the fixed point from here on (never, with a variable speed)

    // prefetch (nseg == 1): cell c of slot s of this thread; cells [0, NV): prev, [NV, 2 NV): cur, (VAR: [2 NV, 3 NV): cs,)
    // last: neighbour of the warp
    constexpr int CELLS = (VAR ? 3 : 2) * NV + 1;
    const bool pre = a.nseg == 1;
    auto cell = [&](int slot, int c) -> unsigned char* {
        return ex_smem + ((static_cast<size_t>(slot) * CELLS + c) * EX_NT + threadIdx.x) * 16;
    };
    const int q0 = (gw * 32 + lane) * U;          // this thread's first point (nseg == 1)
    auto prefetch = [&](int base_n, int slot) {
        const int jn = base_n + group;
        if (pre && jn < a.nlines && q0 < a.pitch) {
            const long long rn = static_cast<long long>(jn) * a.pitch + q0;
#pragma unroll
            for (int c = 0; c < NV; ++c) {
                if (!one) cp_async16(cell(slot, c), prev + rn + c * V);
                cp_async16(cell(slot, NV + c), cur + rn + c * V);
                if constexpr (VAR) cp_async16(cell(slot, 2 * NV + c), csf + rn + c * V);
            }
            if (!one && lane == 0 && q0 > 0) cp_async_small<sizeof(T)>(cell(slot, CELLS - 1), prev + rn - 1);
            if (!one && lane == 31 && q0 + U < a.pitch) cp_async_small<sizeof(T)>(cell(slot, CELLS - 1), prev + rn + U);
        }
        cp_async_commit();
    };
    int it = 0;
    prefetch(blockIdx.x * ngroups, 0);

    for (int base = blockIdx.x * ngroups; base < a.nlines; base += gridDim.x * ngroups, ++it) {
        const int j = base + group;
        const bool live = j < a.nlines;           // (a dead group still walks through the barriers)
        const long long ro = static_cast<long long>(live ? j : 0) * a.pitch;
        const bool src_row = src != nullptr && live && j >= a.sl0 && j < a.sl0 + a.snl;
        T carry = T(0);
        T y[U], cp[U], iv[U];
        for (int s = 0; s < a.nseg; ++s) {
            const int p0 = s * seg_pts + (gw * 32 + lane) * U;
            const int w0 = s * seg_pts + gw * 32 * U;                  // first point of this warp
            const bool fast = live && w0 >= pc && w0 + 32 * U <= n;     // 32 whole stationary units (warp-uniform)
            if (!VAR && !fast) pivots(p0, cp, iv);
            T wp[U], wc[U];
            [[maybe_unused]] T wa[U];                   // VAR: cs, then a_p = ap cs_p
#pragma unroll
            for (int e = 0; e < U; ++e) wp[e] = wc[e] = wa[e] = T(0);
            const bool inrow = live && p0 < a.pitch;   // (pad columns inside the pitch are zero)
            T edge = T(0);                              // lane 0: the point before the warp's first, lane 31: after its last
            if (pre) {
                prefetch(base + gridDim.x * ngroups, (it & 1) ^ 1);   // the next pass, while this one is solved
                cp_async_wait<1>();                                    // this pass's own copies have landed
                if (inrow) {
#pragma unroll
                    for (int c = 0; c < NV; ++c) {
                        if (!one) ld16(reinterpret_cast<const T*>(cell(it & 1, c)), wp + c * V);
                        ld16(reinterpret_cast<const T*>(cell(it & 1, NV + c)), wc + c * V);
                        if constexpr (VAR) ld16(reinterpret_cast<const T*>(cell(it & 1, 2 * NV + c)), wa + c * V);
                    }
                    if (!one && ((lane == 0 && p0 > 0) || (lane == 31 && p0 + U < a.pitch)))
                        edge = *reinterpret_cast<const T*>(cell(it & 1, CELLS - 1));
                }
            } else if (inrow) {
#pragma unroll
                for (int c = 0; c < NV; ++c) {
                    if (!one) ld16(prev + ro + p0 + c * V, wp + c * V);
                    ld16(cur + ro + p0 + c * V, wc + c * V);
                    if constexpr (VAR) ld16(csf + ro + p0 + c * V, wa + c * V);
                }
                if (!one && lane == 0 && p0 > 0) edge = prev[ro + p0 - 1];
                if (!one && lane == 31 && p0 + U < a.pitch) edge = prev[ro + p0 + U];
            }
            if (one) {
#pragma unroll
                for (int e = 0; e < U; ++e) y[e] = wc[e];
            } else {
                T wl = __shfl_up_sync(FULL, wp[U - 1], 1), wr = __shfl_down_sync(FULL, wp[0], 1);
                if (lane == 0) wl = edge;
                if (lane == 31) wr = edge;
#pragma unroll
                for (int e = 0; e < U; ++e) {     // A1: right-hand side of (2.11)
                    const T left = e == 0 ? wl : wp[e - 1], right = e == U - 1 ? wr : wp[e + 1];
                    if constexpr (VAR) {           // am_p = am cs_p at the point of the equation
                        const T amp = am * wa[e];
                        y[e] = fmaT(g2, wc[e], fmaT(amp, left + right, -fmaT(T(2), amp, gam) * wp[e]));
                    } else {
                        y[e] = fmaT(g2, wc[e], fmaT(am, left + right, c1 * wp[e]));
                    }
                }
                if (src_row && p0 < a.sp0 + a.snp && p0 + U > a.sp0) {
#pragma unroll
                    for (int e = 0; e < U; ++e) {
                        const int ps = p0 + e - a.sp0;
                        if (ps >= 0 && ps < a.snp) y[e] = fmaT(q, src[static_cast<size_t>(ps) * a.snl + (j - a.sl0)], y[e]);
                    }
                }
            }
            if constexpr (VAR) {                   // this line's own pivots (host: nseg == 1 with a variable speed)
#pragma unroll
                for (int e = 0; e < U; ++e) wa[e] = p0 + e < n ? ap * wa[e] : T(0);
                group_pivots<T, U>(wa, gam, cp, iv, T(0), wpc, gw, lane, &s_mob[pp][0][group * wpc],
                                   &s_mob[pp][1][group * wpc], &s_mob[pp][2][group * wpc]);
                pp ^= 1;
            }
            carry = group_forward<T, U>(fast, y, cp, iv, S, carry, wpc, gw, lane, &s_agg[pf][0][group * wpc],
                                        &s_agg[pf][1][group * wpc]);
            pf ^= 1;
            if (a.nseg > 1) {
#pragma unroll
                for (int e = 0; e < U; ++e) s_line[static_cast<size_t>(p0 + e)] = y[e];   // parked until the way back
            }
        }
        carry = T(0);
        for (int s = a.nseg - 1; s >= 0; --s) {
            const int p0 = s * seg_pts + (gw * 32 + lane) * U;
            const int w0 = s * seg_pts + gw * 32 * U;
            const bool fast = live && w0 >= pc && w0 + 32 * U <= n;
            if (a.nseg > 1) {
                if (!fast) pivots(p0, cp, iv);
#pragma unroll
                for (int e = 0; e < U; ++e) y[e] = s_line[static_cast<size_t>(p0 + e)];
            }
            carry = group_backward<T, U>(fast, y, cp, S, carry, wpc, gw, lane, &s_agg[pb][2][group * wpc],
                                         &s_agg[pb][3][group * wpc]);
            pb ^= 1;
            if (live && p0 < a.pitch) {
#pragma unroll
                for (int c = 0; c < NV; ++c) st16g(out + ro + p0 + c * V, y + c * V);
            }
        }
    }
}

// ---- y half-step: (A3 + A4) exact ------------------------------------------------------------------------------
// A strip: columns [c0, c0 + sc) over all n rows.  Shared memory: strip[sc][units * (U + 1)] (a unit of U rows is U + 1
// apart: a warp reading one row offset of 32 consecutive units touches 32 distinct bank pairs).
// VAR: a second strip holds a_p = ap cs_p (the solve needs it along the column), so strips are half as wide.
template <typename T, bool VAR>
__global__ void __launch_bounds__(EX_NT) wave2d_exact_y(const __grid_constant__ ExactArgs a)
{
    constexpr int U = EX_U, V = 16 / (int)sizeof(T);
    extern __shared__ __align__(16) unsigned char ex_smem[];
    T* const strip = reinterpret_cast<T*>(ex_smem);
    __shared__ T s_agg[2][4][EX_NW];   // double-buffered like in wave2d_exact_x
    __shared__ T s_mob[VAR ? 2 : 1][3][EX_NW];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wpc = a.wpc, group = warp / wpc, gw = warp % wpc, ngroups = EX_NW / wpc;
    const int nh = a.n_off + 2 * (*a.d_k);
    const Roles R = roles_of(nh, a.fs.ring);
    const T* const prev = static_cast<const T*>(a.fs.b[R.prev]);
    const T* const cur = static_cast<const T*>(a.fs.b[R.cur]);
    T* const out = static_cast<T*>(a.fs.b[R.out]);
    const double* row = a.table + static_cast<size_t>(a.period ? nh % a.period : nh) * ROW_DOUBLES;
    const T am = static_cast<T>(row[ROW_AM]), q = static_cast<T>(row[ROW_Q]), c1 = static_cast<T>(row[ROW_C1]);
    const T g2 = static_cast<T>(a.g2);
    const bool one = a.one != 0;
    const int n = a.n, sc = a.sc;
    const int units = (n + U - 1) / U, cpitch = units * (U + 1);   // strip pitch per column
    const int seg_units = wpc * 32, nseg = (units + seg_units - 1) / seg_units;
    const T* const src = static_cast<const T*>(a.src);
    int pf = 0, pb = 0;
    [[maybe_unused]] int pp = 0;
    Stat<T, U> S;
    S.init(row[ROW_RHO], row[ROW_INV], lane);
    const int pc = VAR ? 0x7fffffff : *a.conv;
    [[maybe_unused]] const T* const csf = static_cast<const T*>(a.cs);
    [[maybe_unused]] const T ap = static_cast<T>(row[ROW_AP]), gam = static_cast<T>(a.gamma);
    [[maybe_unused]] T* const strip_a = strip + static_cast<size_t>(sc) * cpitch;   // VAR: a_p, same layout
    const int ve = sc < V ? sc : V;                  // elements a loader thread moves per access
    const int kcn = sc / ve;                         // accesses per strip row

    for (int c0 = blockIdx.x * sc; c0 < a.nlines; c0 += gridDim.x * sc) {
        // ---- A3: right-hand side of (2.12), assembled by coalesced loads into the strip
        // (batches of UN accesses per thread, all loads of a batch issued before the first use: the fill runs at the
        // memory system's rate, not at one round trip per row)
        constexpr int UN = 4;
        const int total = n * kcn;
        for (int i0 = threadIdx.x; i0 < total; i0 += EX_NT * UN) {
            T vc[UN][V], vm[UN][V], vu[UN][V], vd[UN][V];
            [[maybe_unused]] T vs[UN][V];
#pragma unroll
            for (int k = 0; k < UN; ++k) {
#pragma unroll
                for (int e = 0; e < V; ++e) vc[k][e] = vm[k][e] = vu[k][e] = vd[k][e] = vs[k][e] = T(0);
                const int idx = i0 + k * EX_NT;
                if (idx < total) {
                    const int r = idx / kcn, kc = idx % kcn;
                    const long long o = static_cast<long long>(r) * a.pitch + c0 + kc * ve;   // inside the pitch (pad columns are zero)
                    if constexpr (VAR) {
                        if (ve == V) ld16(csf + o, vs[k]);
                        else
                            for (int e = 0; e < ve; ++e) vs[k][e] = csf[o + e];
                    }
                    if (ve == V) {
                        ld16(cur + o, vc[k]);
                        if (!one) {
                            ld16(prev + o, vm[k]);
                            if (r > 0) ld16(prev + o - a.pitch, vu[k]);
                            if (r + 1 < n) ld16(prev + o + a.pitch, vd[k]);
                        }
                    } else {
                        for (int e = 0; e < ve; ++e) {
                            vc[k][e] = cur[o + e];
                            if (!one) {
                                vm[k][e] = prev[o + e];
                                if (r > 0) vu[k][e] = prev[o + e - a.pitch];
                                if (r + 1 < n) vd[k][e] = prev[o + e + a.pitch];
                            }
                        }
                    }
                }
            }
#pragma unroll
            for (int k = 0; k < UN; ++k) {
                const int idx = i0 + k * EX_NT;
                if (idx < total) {
                    const int r = idx / kcn, kc = idx % kcn;
                    const bool src_r = src != nullptr && !one && r >= a.sp0 && r < a.sp0 + a.snp;
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        if (e < ve) {
                            const int col = c0 + kc * ve + e;
                            T rv;
                            if constexpr (VAR) {   // am_p = am cs_p at the point of the equation
                                const T amp = am * vs[k][e];
                                rv = fmaT(g2, vc[k][e], fmaT(amp, vu[k][e] + vd[k][e], -fmaT(T(2), amp, gam) * vm[k][e]));
                                strip_a[(kc * ve + e) * cpitch + r + r / U] = ap * vs[k][e];
                            } else {
                                rv = one ? vc[k][e] : fmaT(g2, vc[k][e], fmaT(am, vu[k][e] + vd[k][e], c1 * vm[k][e]));
                            }
                            if (src_r && col >= a.sl0 && col < a.sl0 + a.snl)
                                rv = fmaT(q, src[static_cast<size_t>(r - a.sp0) * a.snl + (col - a.sl0)], rv);
                            strip[(kc * ve + e) * cpitch + r + r / U] = rv;
                        }
                    }
                }
            }
        }
        __syncthreads();
        // ---- A4: the columns of the strip, ngroups at a time, in place
        for (int cb = 0; cb < sc; cb += ngroups) {
            const int col = cb + group;
            const bool live = col < sc;
            T* const line = strip + static_cast<size_t>(live ? col : 0) * cpitch;
            T carry = T(0);
            T y[U], cp[U], iv[U];
            for (int s = 0; s < nseg; ++s) {
                const int u = s * seg_units + gw * 32 + lane, p0 = u * U;
                const int w0 = (s * seg_units + gw * 32) * U;
                const bool fast = live && w0 >= pc && w0 + 32 * U <= n;
#pragma unroll
                for (int e = 0; e < U; ++e) {
                    const bool in = live && p0 + e < n;
                    if (!VAR && !fast) {
                        cp[e] = p0 + e < n ? static_cast<T>(a.cpv[p0 + e]) : T(0);
                        iv[e] = p0 + e < n ? static_cast<T>(a.ivv[p0 + e]) : T(0);
                    }
                    y[e] = in ? line[u * (U + 1) + e] : T(0);
                }
                if constexpr (VAR) {               // this column's own pivots (host: nseg == 1 with a variable speed)
                    T wa[U];
#pragma unroll
                    for (int e = 0; e < U; ++e)
                        wa[e] = live && p0 + e < n ? strip_a[static_cast<size_t>(col) * cpitch + u * (U + 1) + e] : T(0);
                    group_pivots<T, U>(wa, gam, cp, iv, T(0), wpc, gw, lane, &s_mob[pp][0][group * wpc],
                                       &s_mob[pp][1][group * wpc], &s_mob[pp][2][group * wpc]);
                    pp ^= 1;
                }
                carry = group_forward<T, U>(fast, y, cp, iv, S, carry, wpc, gw, lane, &s_agg[pf][0][group * wpc],
                                            &s_agg[pf][1][group * wpc]);
                pf ^= 1;
                if (nseg > 1 && live) {
#pragma unroll
                    for (int e = 0; e < U; ++e)
                        if (p0 + e < n) line[u * (U + 1) + e] = y[e];
                }
            }
            carry = T(0);
            for (int s = nseg - 1; s >= 0; --s) {
                const int u = s * seg_units + gw * 32 + lane, p0 = u * U;
                const int w0 = (s * seg_units + gw * 32) * U;
                const bool fast = live && w0 >= pc && w0 + 32 * U <= n;
                if (nseg > 1) {
#pragma unroll
                    for (int e = 0; e < U; ++e) {
                        if (!fast) cp[e] = p0 + e < n ? static_cast<T>(a.cpv[p0 + e]) : T(0);
                        y[e] = live && p0 + e < n ? line[u * (U + 1) + e] : T(0);
                    }
                }
                carry = group_backward<T, U>(fast, y, cp, S, carry, wpc, gw, lane, &s_agg[pb][2][group * wpc],
                                             &s_agg[pb][3][group * wpc]);
                pb ^= 1;
                if (live) {
#pragma unroll
                    for (int e = 0; e < U; ++e)
                        if (p0 + e < n) line[u * (U + 1) + e] = y[e];
                }
            }
        }
        __syncthreads();
        // ---- coalesced stores of the strip
        for (int idx = threadIdx.x; idx < n * kcn; idx += EX_NT) {
            const int r = idx / kcn, kc = idx % kcn;
            T* const o = out + static_cast<long long>(r) * a.pitch + c0 + kc * ve;
            T vo[V];
#pragma unroll
            for (int e = 0; e < V; ++e) vo[e] = e < ve ? strip[(kc * ve + e) * cpitch + r + r / U] : T(0);
            if (ve == V) st16g(o, vo);
            else
                for (int e = 0; e < ve; ++e) o[e] = vo[e];
        }
        __syncthreads();   // the strip is refilled by the next pass
    }
}

}  // namespace w2d
