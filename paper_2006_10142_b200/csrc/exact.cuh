// exact.cuh -- the untruncated line solvers (solver EXACT): any tau / h, any line length up to 16384 unknowns.
//
// The north_star's solver sketch -- a line "staged whole in shared memory ... solved by cyclic reduction (or PCR
// for the last levels) with warp shuffles" (CRM_forward, cr_div, CRM_backward) -- with the
// changes the scalar coefficients allow:
//   * register blocking: a thread owns U = 8 consecutive points and eliminates them serially (the first log2 U
//     reduction levels happen in registers, no strided shared-memory access, no bank conflicts);
//   * the remaining levels are a scan: both elimination sweeps are first-order linear recurrences, so the carries
//     between units follow from the inclusive scan of the pairs (A, L) -> (A A', L + A L') -- five shuffle rounds inside
//     a warp, one more scan over the warp aggregates of the line in shared memory.  That is the log2(n+1) - 1 levels
//     of P:124-128 with 2 barriers (of the line's warps) per sweep direction;
//   * Toeplitz systems (c = c(t)) run the recurrences with the STATIONARY factors everywhere (cp = rho,
//     inv = 1 / (beta - ap rho): the exact LU of the matrix whose first diagonal entry is beta - ap rho instead of beta),
//     on the line padded to whole warps, and repair both ends afterwards: the difference to the true solution solves
//     the homogeneous recurrence, so it is  A rho^(p+1) + B rho^(n-p)  with two scalars per line that follow from the
//     first value and the value at index n of the stationary solution (see boundary_scalars).  No pivot arrays, no
//     per-point coefficients, the scan carries values only; exact to rounding for every tau / h.
//   * a variable speed c(t) cs(x,y) (VAR) keeps per-point pivots: a scan of linear-fractional maps (group_pivots).
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
// y strips: elements between the columns of a strip -- a unit of U rows is U + 1 apart (a warp reading one row offset of 32
// consecutive units touches 32 distinct banks), made odd so that the columns of a row do not share a bank either
__host__ __device__ constexpr int ex_cpitch(int units) { return (units * (EX_U + 1)) | 1; }

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
        double al = 1.0, ar = 1.0, Ad = pw[U - 1];    // A^lane, A^(31 - lane) by binary powering
#pragma unroll
        for (int d = 0; d < 5; ++d, Ad *= Ad) {
            if ((lane >> d) & 1) al *= Ad;
            if (((31 - lane) >> d) & 1) ar *= Ad;
        }
        Alane = static_cast<T>(al);
        Arev = static_cast<T>(ar);
    }
};

// The two ends of a Toeplitz line.  x'' = the stationary recurrences run over the padded line (x''_{npad} = 0).  The true
// solution x (x_{-1} = x_n = 0, true first pivot) differs from it by a solution of the homogeneous recurrence,
//      x_p = x''_p - A rho^(p+1) - B rho^(n-p),       0 <= p < n,
// and the first and last equation of the line give, with eps = rho^(n+1),
//      A + B eps = rho x''_0 ,     A eps + B = x''_n        (x''_n := 0 if the padded line ends at n).
template <typename T>
struct Ends {
    double lnr, rho, eps, den;     // ln rho, rho, rho^(n+1), 1 / (1 - eps^2)
    __device__ __forceinline__ void init(double rho_d, double ln_rho, int n)
    {
        rho = rho_d;
        lnr = ln_rho;
        eps = exp((n + 1) * lnr);
        den = 1.0 / (1.0 - eps * eps);
    }
    __device__ __forceinline__ T power(int k) const   // rho^k, 0 where it is below every rounding unit that matters
    {
        const double x = k * lnr;
        return x < -96.0 ? T(0) : static_cast<T>(exp(x));
    }
    __device__ __forceinline__ void scalars(T x0, T xn, T& A, T& B) const
    {
        const double a = (rho * static_cast<double>(x0) - eps * static_cast<double>(xn)) * den;
        const double b = (static_cast<double>(xn) - eps * rho * static_cast<double>(x0)) * den;
        A = static_cast<T>(a);
        B = static_cast<T>(b);
    }
};
// x[e] -= A rho^(p0+e+1) + B rho^(n-p0-e) for the points of a unit that lie on the line (m = n - p0 of them, if fewer
// than U); PA = rho^(p0+1), PB = rho^(m-U+1) (Ends::power; unused in the unit that holds the end of the line, which
// reads rho^(m-e) from the table spw[k] = rho^(k+1) in shared memory).  Points beyond the line are set to 0.
template <typename T, int U>
__device__ __forceinline__ void repair_unit(T (&x)[U], const Stat<T, U>& S, T A, T B, T PA, T PB, int m, const T* spw)
{
    const T a = A * PA;
    if (m >= U) {
        const T b = B * PB;
        if (a == T(0) && b == T(0)) return;
#pragma unroll
        for (int e = 0; e < U; ++e) {
            const T fa = e == 0 ? T(1) : S.pw[e - 1], fb = e == U - 1 ? T(1) : S.pw[U - 2 - e];
            x[e] -= fmaT(a, fa, b * fb);
        }
    } else {
#pragma unroll
        for (int e = 0; e < U; ++e) {
            const T fa = e == 0 ? T(1) : S.pw[e - 1];
            x[e] = e < m ? x[e] - fmaT(a, fa, B * spw[m - e - 1]) : T(0);
        }
    }
}

// The warps of one line synchronise among themselves only (hardware barriers 1..8: wpc >= 2 means at most 8 groups),
// so the lines a CTA works on at the same time do not wait for one another.
__device__ __forceinline__ void group_sync(int group, int wpc)
{
    if (wpc > 1) named_bar_sync(1 + group, 32 * wpc);
    else __syncwarp();
}

// ---- block-wide solve of one line segment ------------------------------------------------------------------
// A "group" is wpc consecutive warps of the CTA; thread (gw, lane) of the group owns unit gw * 32 + lane of the segment.
// sA, sL (forward) and sB, sH (backward) are the group's slices [wpc] of the CTA's aggregate arrays.  Every thread of
// a group must call these (they contain one barrier of the group each).

// General coefficients (variable speed): cp[], iv[] are this unit's pivots.
// y[] holds r on entry and the true y on exit.  cin: y just before the segment.  Returns y at the end of the segment.
template <typename T, int U>
__device__ __forceinline__ T group_forward(T (&y)[U], const T (&cp)[U], const T (&iv)[U], T cin, int wpc, int gw, int lane,
                                           T* sA, T* sL, int group)
{
    constexpr unsigned FULL = 0xffffffffu;
    T a = T(1), v = T(0);
#pragma unroll
    for (int e = 0; e < U; ++e) {
        v = fmaT(cp[e], v, y[e] * iv[e]);
        y[e] = v;
        a *= cp[e];
    }
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const T a2 = __shfl_up_sync(FULL, a, d), v2 = __shfl_up_sync(FULL, v, d);
        if (lane >= d) {
            v = fmaT(a, v2, v);
            a *= a2;
        }
    }
    if (lane == 31) {
        sA[gw] = a;
        sL[gw] = v;
    }
    group_sync(group, wpc);
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
    const T pv = __shfl_up_sync(FULL, v, 1), pa = __shfl_up_sync(FULL, a, 1);
    T c = lane == 0 ? cw : fmaT(pa, cw, pv);
#pragma unroll
    for (int e = 0; e < U; ++e) {
        c *= cp[e];
        y[e] += c;
    }
    return cout;
}

// y[] holds the true y on entry and x on exit.  xin: x just after the segment.  Returns x at the start of the segment.
template <typename T, int U>
__device__ __forceinline__ T group_backward(T (&y)[U], const T (&cp)[U], T xin, int wpc, int gw, int lane, T* sB, T* sH,
                                            int group)
{
    constexpr unsigned FULL = 0xffffffffu;
    T a = cp[U - 1];
#pragma unroll
    for (int e = U - 2; e >= 0; --e) {
        y[e] = fmaT(cp[e], y[e + 1], y[e]);
        a *= cp[e];
    }
    T v = y[0];
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const T a2 = __shfl_down_sync(FULL, a, d), v2 = __shfl_down_sync(FULL, v, d);
        if (lane + d < 32) {
            v = fmaT(a, v2, v);
            a *= a2;
        }
    }
    if (lane == 0) {
        sB[gw] = a;
        sH[gw] = v;
    }
    group_sync(group, wpc);
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
    const T nv = __shfl_down_sync(FULL, v, 1), na = __shfl_down_sync(FULL, a, 1);
    T c = lane == 31 ? xw : fmaT(na, xw, nv);
#pragma unroll
    for (int e = U - 1; e >= 0; --e) {
        c *= cp[e];
        y[e] += c;
    }
    return cout;
}

// ---- the stationary recurrences (Toeplitz lines) --------------------------------------------------------------
// Every unit has cp = rho, inv constant, A = rho^U: the scans carry values only.  Inside a warp five shuffle rounds with the
// constant factors A^(2^d); across the warps of the line a Horner loop over the warp aggregates in shared memory
// (W = A^32 per warp).  y[] holds r on entry and the true y on exit; cin: y just before the segment; returns y at the end of
// the segment (only if `chain`: a further segment follows).
template <typename T, int U>
__device__ __forceinline__ T stat_forward(T (&y)[U], const Stat<T, U>& S, T cin, int wpc, int gw, int lane, T* sL, int group,
                                          bool chain)
{
    constexpr unsigned FULL = 0xffffffffu;
    T f = y[0] * S.inv;
    y[0] = f;
#pragma unroll
    for (int e = 1; e < U; ++e) {
        f = fmaT(S.rho, f, y[e] * S.inv);
        y[e] = f;
    }
    T v = f;
#pragma unroll
    for (int d = 0; d < 5; ++d) {
        const T v2 = __shfl_up_sync(FULL, v, 1 << d);
        if (lane >= (1 << d)) v = fmaT(S.Ap[d], v2, v);
    }
    T cw = cin, cout = T(0);
    if (wpc > 1) {
        if (lane == 31) sL[gw] = v;
        group_sync(group, wpc);
        for (int j = 0; j < gw; ++j) cw = fmaT(S.Ap[5], cw, sL[j]);      // y entering this warp
        if (chain) {
            cout = cw;
            for (int j = gw; j < wpc; ++j) cout = fmaT(S.Ap[5], cout, sL[j]);
        }
    } else if (chain) {
        cout = fmaT(S.Ap[5], cin, __shfl_sync(FULL, v, 31));
    }
    const T pv = __shfl_up_sync(FULL, v, 1);
    const T c = lane == 0 ? cw : fmaT(S.Alane, cw, pv);   // y at the end of the previous unit
#pragma unroll
    for (int e = 0; e < U; ++e) y[e] = fmaT(S.pw[e], c, y[e]);
    return cout;
}

// y[] holds the true y on entry and x on exit.  xin: x just after the segment.  Returns x at the start of the segment.
template <typename T, int U>
__device__ __forceinline__ T stat_backward(T (&y)[U], const Stat<T, U>& S, T xin, int wpc, int gw, int lane, T* sH, int group,
                                           bool chain)
{
    constexpr unsigned FULL = 0xffffffffu;
#pragma unroll
    for (int e = U - 2; e >= 0; --e) y[e] = fmaT(S.rho, y[e + 1], y[e]);
    T v = y[0];
#pragma unroll
    for (int d = 0; d < 5; ++d) {
        const T v2 = __shfl_down_sync(FULL, v, 1 << d);
        if (lane + (1 << d) < 32) v = fmaT(S.Ap[d], v2, v);
    }
    T xw = xin, cout = T(0);
    if (wpc > 1) {
        if (lane == 0) sH[gw] = v;
        group_sync(group, wpc);
        for (int j = wpc - 1; j > gw; --j) xw = fmaT(S.Ap[5], xw, sH[j]);   // x entering this warp from the right
        if (chain) {
            cout = xw;
            for (int j = gw; j >= 0; --j) cout = fmaT(S.Ap[5], cout, sH[j]);
        }
    } else if (chain) {
        cout = fmaT(S.Ap[5], xin, __shfl_sync(FULL, v, 0));
    }
    const T nv = __shfl_down_sync(FULL, v, 1);
    const T c = lane == 31 ? xw : fmaT(S.Arev, xw, nv);   // x at the start of the next unit
#pragma unroll
    for (int e = 0; e < U; ++e) y[e] = fmaT(S.pw[U - 1 - e], c, y[e]);
    return cout;
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
                                          int lane, T* sMA, T* sMB, T* sMC, int group)
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
    group_sync(group, wpc);
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
__device__ __forceinline__ T ld1(const T* p)
{
    return *p;
}
template <typename T>
__device__ __forceinline__ void st16g(T* p, const T* v)
{
    if constexpr (sizeof(T) == 8) *reinterpret_cast<double2*>(p) = make_double2(v[0], v[1]);
    else *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
}

// per-thread asynchronous copies global -> shared (LDGSTS, through L2 only): a thread prefetches its own points of
// the next row
__device__ __forceinline__ void cp_async16(void* dst, const void* src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Scratch of the block-wide scans, double-buffered: consecutive forward (or backward) calls of a group alternate, so a
// warp that runs ahead into the next call never overwrites what a slower warp still reads (one barrier per call).
template <typename T>
struct ExactScratch {
    T agg[2][4][EX_NW];
    T mob[2][3][EX_NW];   // aggregates of the pivot scan (VAR), double-buffered likewise
    T ends[EX_NW][2];     // per group: x''_0 and x''_n of its line (Toeplitz lines, see Ends)
    T pw[EX_NW][EX_U];    // per group: rho^(k+1)
};

// ---- x half-step: (A1 + A2) exact ------------------------------------------------------------------------------
// The CTAs loop over passes of EX_NW / wpc rows.  Dynamic shared memory:
//   nseg == 1: two prefetch slots of EX_NT * (2 NV + 1) 16-byte cells -- while a pass is solved, every thread's own
//              points of the next pass's row (and the two neighbour values of a warp) are already on their way;
//   nseg  > 1: the parked line, nseg * wpc * 32 * U values (no prefetch: the line itself fills shared memory).
// VAR: variable speed -- one more field (cs) per row, the pivots come from group_pivots, no stationary path.
// SEG1: compiled for lines of one segment (n <= 4096: the segment loops, the parked line and their tests fold away).
template <typename T, bool VAR, bool SEG1>
__device__ __forceinline__ void exact_x_half_step(const ExactArgs& a, int nh, unsigned char* ex_smem, ExactScratch<T>& sc_)
{
    constexpr int U = EX_U, V = 16 / (int)sizeof(T), NV = U / V;
    constexpr unsigned FULL = 0xffffffffu;
    T* const s_line = reinterpret_cast<T*>(ex_smem);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wpc = a.wpc, group = warp / wpc, gw = warp % wpc, ngroups = EX_NW / wpc;
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
    const int nseg = SEG1 ? 1 : a.nseg;
    const int n = a.n, seg_pts = wpc * 32 * U, npad = nseg * seg_pts;
    const T* const src = static_cast<const T*>(a.src);
    int pf = 0, pb = 0;   // buffer parity of the next forward / backward call
    [[maybe_unused]] int pp = 0;

    Stat<T, U> S;
    S.init(row[ROW_RHO], row[ROW_INV], lane);
    [[maybe_unused]] Ends<T> E;
    [[maybe_unused]] T PA = T(0), PB = T(0);      // nseg == 1: this thread's rho^(p0+1), rho^(n-p0-U+1)
    [[maybe_unused]] T* const s_ends = sc_.ends[group];
    [[maybe_unused]] const T* const s_pw = sc_.pw[group];
    if constexpr (!VAR) {
        E.init(row[ROW_RHO], row[ROW_LNR], n);
        if (gw == 0 && lane == 0) {
#pragma unroll
            for (int e = 0; e < U; ++e) sc_.pw[group][e] = S.pw[e];
        }
        const int p0 = (gw * 32 + lane) * U;
        if (nseg == 1 && p0 < n) {
            PA = E.power(p0 + 1);
            if (n - p0 >= U) PB = E.power(n - p0 - U + 1);
        }
    }

    // prefetch (nseg == 1): cell c of slot s of this thread; cells [0, NV): prev, [NV, 2 NV): cur, (VAR: [2 NV, 3 NV): cs,)
    // last: the 16 bytes of prev next to the warp (lane 0: before its first point, lane 31: after its last)
    constexpr int CELLS = (VAR ? 3 : 2) * NV + 1;
    const bool pre = nseg == 1;
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
            if (!one && lane == 0 && q0 > 0) cp_async16(cell(slot, CELLS - 1), prev + rn - V);
            if (!one && lane == 31 && q0 + U < a.pitch) cp_async16(cell(slot, CELLS - 1), prev + rn + U);
        }
        cp_async_commit();
    };
    int it = 0;
    prefetch(blockIdx.x * ngroups, 0);

    for (int base = blockIdx.x * ngroups; base < a.nlines; base += gridDim.x * ngroups, ++it) {
        const int j = base + group;
        const bool live = j < a.nlines;           // (a dead group still walks through its barriers)
        const long long ro = static_cast<long long>(live ? j : 0) * a.pitch;
        const bool src_row = src != nullptr && live && j >= a.sl0 && j < a.sl0 + a.snl;
        T carry = T(0);
        T y[U];
        [[maybe_unused]] T cp[VAR ? U : 1], iv[VAR ? U : 1];
        for (int s = 0; s < nseg; ++s) {
            const int p0 = s * seg_pts + (gw * 32 + lane) * U;
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
                    if (!one && lane == 0 && p0 > 0) edge = reinterpret_cast<const T*>(cell(it & 1, CELLS - 1))[V - 1];
                    if (!one && lane == 31 && p0 + U < a.pitch) edge = reinterpret_cast<const T*>(cell(it & 1, CELLS - 1))[0];
                }
            } else if (inrow) {
#pragma unroll
                for (int c = 0; c < NV; ++c) {
                    if (!one) ld16(prev + ro + p0 + c * V, wp + c * V);
                    ld16(cur + ro + p0 + c * V, wc + c * V);
                    if constexpr (VAR) ld16(csf + ro + p0 + c * V, wa + c * V);
                }
                if (!one && lane == 0 && p0 > 0) edge = ld1(prev + ro + p0 - 1);
                if (!one && lane == 31 && p0 + U < a.pitch) edge = ld1(prev + ro + p0 + U);
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
                group_pivots<T, U>(wa, gam, cp, iv, T(0), wpc, gw, lane, &sc_.mob[pp][0][group * wpc],
                                   &sc_.mob[pp][1][group * wpc], &sc_.mob[pp][2][group * wpc], group);
                pp ^= 1;
                carry = group_forward<T, U>(y, cp, iv, carry, wpc, gw, lane, &sc_.agg[pf][0][group * wpc],
                                                        &sc_.agg[pf][1][group * wpc], group);
            } else {                               // Toeplitz: stationary factors on the padded line (see Ends)
                carry = stat_forward<T, U>(y, S, carry, wpc, gw, lane, &sc_.agg[pf][1][group * wpc], group, nseg > 1);
            }
            pf ^= 1;
            if (nseg > 1) {
#pragma unroll
                for (int e = 0; e < U; ++e) s_line[static_cast<size_t>(p0 + e)] = y[e];   // parked until the way back
            }
        }
        carry = T(0);
        for (int s = nseg - 1; s >= 0; --s) {
            const int p0 = s * seg_pts + (gw * 32 + lane) * U;
            if (nseg > 1) {
#pragma unroll
                for (int e = 0; e < U; ++e) y[e] = s_line[static_cast<size_t>(p0 + e)];
            }
            if constexpr (VAR) {
                carry = group_backward<T, U>(y, cp, carry, wpc, gw, lane, &sc_.agg[pb][2][group * wpc],
                                                         &sc_.agg[pb][3][group * wpc], group);
                pb ^= 1;
                if (live && p0 < a.pitch) {
#pragma unroll
                    for (int c = 0; c < NV; ++c) st16g(out + ro + p0 + c * V, y + c * V);
                }
            } else {
                carry = stat_backward<T, U>(y, S, carry, wpc, gw, lane, &sc_.agg[pb][3][group * wpc], group, nseg > 1);
                pb ^= 1;
                if (p0 == 0) s_ends[0] = y[0];                 // x''_0
                if (p0 <= n && n < p0 + U) {                   // x''_n (nobody holds it if the padded line ends at n)
                    T xn = y[0];
#pragma unroll
                    for (int e = 1; e < U; ++e) xn = n - p0 == e ? y[e] : xn;
                    s_ends[1] = xn;
                }
                if (nseg > 1) {
#pragma unroll
                    for (int e = 0; e < U; ++e) s_line[static_cast<size_t>(p0 + e)] = y[e];   // x'' until both ends are known
                }
            }
        }
        if constexpr (!VAR) {                      // repair both ends (see Ends), then store
            group_sync(group, wpc);
            T A, B;
            E.scalars(s_ends[0], n < npad ? s_ends[1] : T(0), A, B);
            if (nseg == 1) {
                const int p0 = (gw * 32 + lane) * U;
                repair_unit<T, U>(y, S, A, B, PA, PB, n - p0, s_pw);
                if (live && p0 < a.pitch) {
#pragma unroll
                    for (int c = 0; c < NV; ++c) st16g(out + ro + p0 + c * V, y + c * V);
                }
            } else {
                for (int s = 0; s < nseg; ++s) {
                    const int p0 = s * seg_pts + (gw * 32 + lane) * U, m = n - p0;
#pragma unroll
                    for (int e = 0; e < U; ++e) y[e] = s_line[static_cast<size_t>(p0 + e)];
                    repair_unit<T, U>(y, S, A, B, m > 0 ? E.power(p0 + 1) : T(0), m >= U ? E.power(m - U + 1) : T(0), m, s_pw);
                    if (live && p0 < a.pitch) {
#pragma unroll
                        for (int c = 0; c < NV; ++c) st16g(out + ro + p0 + c * V, y + c * V);
                    }
                }
            }
            if (nseg > 1) group_sync(group, wpc);   // the parked line is rewritten by the next pass
        }
    }
    cp_async_wait<0>();
}

template <typename T, bool VAR, bool SEG1>
__global__ void __launch_bounds__(EX_NT) wave2d_exact_x(const __grid_constant__ ExactArgs a)
{
    extern __shared__ __align__(16) unsigned char ex_smem[];
    __shared__ ExactScratch<T> scratch;
    exact_x_half_step<T, VAR, SEG1>(a, a.n_off + 2 * (*a.d_k), ex_smem, scratch);
}

// ---- y half-step: (A3 + A4) exact ------------------------------------------------------------------------------
// A strip: columns [c0, c0 + sc) over all n rows.  Shared memory: strip[sc][units * (U + 1)] (a unit of U rows is U + 1
// apart: a warp reading one row offset of 32 consecutive units touches 32 distinct bank pairs).
// VAR: a second strip holds a_p = ap cs_p (the solve needs it along the column), so strips are half as wide.
template <typename T, bool VAR, bool SEG1>
__device__ __forceinline__ void exact_y_half_step(const ExactArgs& a, int nh, unsigned char* ex_smem, ExactScratch<T>& sc_)
{
    constexpr int U = EX_U, V = 16 / (int)sizeof(T);
    T* const strip = reinterpret_cast<T*>(ex_smem);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wpc = a.wpc, group = warp / wpc, gw = warp % wpc, ngroups = EX_NW / wpc;
    const Roles R = roles_of(nh, a.fs.ring);
    const T* const prev = static_cast<const T*>(a.fs.b[R.prev]);
    const T* const cur = static_cast<const T*>(a.fs.b[R.cur]);
    T* const out = static_cast<T*>(a.fs.b[R.out]);
    const double* row = a.table + static_cast<size_t>(a.period ? nh % a.period : nh) * ROW_DOUBLES;
    const T am = static_cast<T>(row[ROW_AM]), q = static_cast<T>(row[ROW_Q]), c1 = static_cast<T>(row[ROW_C1]);
    const T g2 = static_cast<T>(a.g2);
    const bool one = a.one != 0;
    const int n = a.n, sc = a.sc;
    static_assert(U == 8, "strip addressing uses r + (r >> 3)");
    const int units = (n + U - 1) / U, cpitch = ex_cpitch(units);   // strip pitch per column
    const int seg_units = wpc * 32, nseg = SEG1 ? 1 : (units + seg_units - 1) / seg_units;
    const T* const src = static_cast<const T*>(a.src);
    int pf = 0, pb = 0;
    [[maybe_unused]] int pp = 0;
    Stat<T, U> S;
    S.init(row[ROW_RHO], row[ROW_INV], lane);
    const int npad = nseg * seg_units * U;
    [[maybe_unused]] Ends<T> E;
    [[maybe_unused]] T PA = T(0), PB = T(0);      // nseg == 1: this thread's rho^(p0+1), rho^(n-p0-U+1)
    [[maybe_unused]] T* const s_ends = sc_.ends[group];
    [[maybe_unused]] const T* const s_pw = sc_.pw[group];
    if constexpr (!VAR) {
        E.init(row[ROW_RHO], row[ROW_LNR], n);
        if (gw == 0 && lane == 0) {
#pragma unroll
            for (int e = 0; e < U; ++e) sc_.pw[group][e] = S.pw[e];
        }
        const int p0 = (gw * 32 + lane) * U;
        if (nseg == 1 && p0 < n) {
            PA = E.power(p0 + 1);
            if (n - p0 >= U) PB = E.power(n - p0 - U + 1);
        }
    }
    [[maybe_unused]] const T* const csf = static_cast<const T*>(a.cs);
    [[maybe_unused]] const T ap = static_cast<T>(row[ROW_AP]), gam = static_cast<T>(a.gamma);
    [[maybe_unused]] T* const strip_a = strip + static_cast<size_t>(sc) * cpitch;   // VAR: a_p, same layout
    const int ve = sc < V ? sc : V;                  // elements a loader thread moves per access
    const int kcn = sc / ve;                         // accesses per strip row (a power of two, at most 8)
    const int lk = 31 - __clz(kcn);

    for (int c0 = blockIdx.x * sc; c0 < a.nlines; c0 += gridDim.x * sc) {
        // ---- A3: right-hand side of (2.12), assembled by coalesced loads into the strip.  A thread takes RB = 4
        // consecutive rows of one 16-byte column chunk: the stencil neighbours of w_{n-1} inside the block are its own
        // registers (6 loads of w_{n-1} for 4 rows), and all loads of a block are issued before the first use.
        // Consecutive lanes take the chunks of a row block, then the next row block.
        constexpr int RB = 4;
        const int items = ((n + RB - 1) / RB) << lk;
        for (int i = threadIdx.x; i < items; i += EX_NT) {
            const int r0 = (i >> lk) * RB, kc = i & (kcn - 1);
            T vc[RB][V], vm[RB + 2][V];
            [[maybe_unused]] T vs[RB][V];
#pragma unroll
            for (int k = 0; k < RB + 2; ++k) {
#pragma unroll
                for (int e = 0; e < V; ++e) {
                    vm[k][e] = T(0);
                    if (k < RB) vc[k][e] = vs[k][e] = T(0);
                }
            }
            const T* const pc_ = cur + static_cast<long long>(r0) * a.pitch + c0 + kc * ve;   // inside the pitch (pad columns are zero)
            const T* const pm_ = prev + static_cast<long long>(r0 - 1) * a.pitch + c0 + kc * ve;
            if (ve == V) {
#pragma unroll
                for (int k = 0; k < RB; ++k) {
                    if (r0 + k < n) {
                        ld16(pc_ + k * a.pitch, vc[k]);
                        if constexpr (VAR) ld16(csf + (pc_ - cur) + k * a.pitch, vs[k]);
                    }
                }
                if (!one) {
#pragma unroll
                    for (int k = 0; k < RB + 2; ++k)
                        if (r0 + k - 1 >= 0 && r0 + k - 1 < n) ld16(pm_ + k * a.pitch, vm[k]);
                }
            } else {
                for (int e = 0; e < ve; ++e) {
#pragma unroll
                    for (int k = 0; k < RB; ++k) {
                        if (r0 + k < n) {
                            vc[k][e] = ld1(pc_ + k * a.pitch + e);
                            if constexpr (VAR) vs[k][e] = ld1(csf + (pc_ - cur) + k * a.pitch + e);
                        }
                    }
                    if (!one) {
#pragma unroll
                        for (int k = 0; k < RB + 2; ++k)
                            if (r0 + k - 1 >= 0 && r0 + k - 1 < n) vm[k][e] = ld1(pm_ + k * a.pitch + e);
                    }
                }
            }
            // (the item's column range and its strip column are fixed: the source test and the strip addresses per item)
            const int colb = c0 + kc * ve;
            const bool src_item = src != nullptr && !one && colb < a.sl0 + a.snl && colb + ve > a.sl0 &&
                                  r0 < a.sp0 + a.snp && r0 + RB > a.sp0;
            T* const sp = strip + static_cast<size_t>(kc * ve) * cpitch;
            [[maybe_unused]] T* const spa = strip_a + static_cast<size_t>(kc * ve) * cpitch;
#pragma unroll
            for (int k = 0; k < RB; ++k) {
                const int r = r0 + k;
                if (r < n) {
                    const int so = r + (r >> 3);
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        if (e < ve) {
                            T rv;
                            if constexpr (VAR) {   // am_p = am cs_p at the point of the equation
                                const T amp = am * vs[k][e];
                                rv = fmaT(g2, vc[k][e], fmaT(amp, vm[k][e] + vm[k + 2][e], -fmaT(T(2), amp, gam) * vm[k + 1][e]));
                                spa[e * cpitch + so] = ap * vs[k][e];
                            } else {
                                rv = one ? vc[k][e] : fmaT(g2, vc[k][e], fmaT(am, vm[k][e] + vm[k + 2][e], c1 * vm[k + 1][e]));
                            }
                            if (src_item) {
                                const int col = colb + e;
                                if (r >= a.sp0 && r < a.sp0 + a.snp && col >= a.sl0 && col < a.sl0 + a.snl)
                                    rv = fmaT(q, src[static_cast<size_t>(r - a.sp0) * a.snl + (col - a.sl0)], rv);
                            }
                            sp[e * cpitch + so] = rv;
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
            T y[U];
            [[maybe_unused]] T cp[VAR ? U : 1], iv[VAR ? U : 1];
            for (int s = 0; s < nseg; ++s) {
                const int u = s * seg_units + gw * 32 + lane, p0 = u * U;
#pragma unroll
                for (int e = 0; e < U; ++e) y[e] = live && p0 + e < n ? line[u * (U + 1) + e] : T(0);
                if constexpr (VAR) {               // this column's own pivots (host: nseg == 1 with a variable speed)
                    T wa[U];
#pragma unroll
                    for (int e = 0; e < U; ++e)
                        wa[e] = live && p0 + e < n ? strip_a[static_cast<size_t>(col) * cpitch + u * (U + 1) + e] : T(0);
                    group_pivots<T, U>(wa, gam, cp, iv, T(0), wpc, gw, lane, &sc_.mob[pp][0][group * wpc],
                                       &sc_.mob[pp][1][group * wpc], &sc_.mob[pp][2][group * wpc], group);
                    pp ^= 1;
                    carry = group_forward<T, U>(y, cp, iv, carry, wpc, gw, lane, &sc_.agg[pf][0][group * wpc],
                                                            &sc_.agg[pf][1][group * wpc], group);
                } else {                           // Toeplitz: stationary factors on the padded line (see Ends)
                    carry = stat_forward<T, U>(y, S, carry, wpc, gw, lane, &sc_.agg[pf][1][group * wpc], group, nseg > 1);
                }
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
                if (nseg > 1) {
#pragma unroll
                    for (int e = 0; e < U; ++e) y[e] = live && p0 + e < n ? line[u * (U + 1) + e] : T(0);
                }
                if constexpr (VAR) {
                    carry = group_backward<T, U>(y, cp, carry, wpc, gw, lane, &sc_.agg[pb][2][group * wpc],
                                                             &sc_.agg[pb][3][group * wpc], group);
                } else {
                    carry = stat_backward<T, U>(y, S, carry, wpc, gw, lane, &sc_.agg[pb][3][group * wpc], group, nseg > 1);
                    if (p0 == 0) s_ends[0] = y[0];             // x''_0
                    if (p0 <= n && n < p0 + U) {               // x''_n (nobody holds it if the padded line ends at n)
                        T xn = y[0];
#pragma unroll
                        for (int e = 1; e < U; ++e) xn = n - p0 == e ? y[e] : xn;
                        s_ends[1] = xn;
                    }
                }
                pb ^= 1;
                if (live && (VAR || nseg > 1)) {   // (Toeplitz, one segment: repaired in registers below)
#pragma unroll
                    for (int e = 0; e < U; ++e)
                        if (p0 + e < n) line[u * (U + 1) + e] = y[e];
                }
            }
            if constexpr (!VAR) {                  // repair both ends (see Ends)
                group_sync(group, wpc);
                T A, B;
                E.scalars(s_ends[0], n < npad ? s_ends[1] : T(0), A, B);
                for (int s = 0; s < nseg; ++s) {
                    const int u = s * seg_units + gw * 32 + lane, p0 = u * U, m = n - p0;
                    if (nseg > 1) {
#pragma unroll
                        for (int e = 0; e < U; ++e) y[e] = live && p0 + e < n ? line[u * (U + 1) + e] : T(0);
                        repair_unit<T, U>(y, S, A, B, m > 0 ? E.power(p0 + 1) : T(0), m >= U ? E.power(m - U + 1) : T(0), m, s_pw);
                    } else {
                        repair_unit<T, U>(y, S, A, B, PA, PB, m, s_pw);
                    }
                    if (live) {
#pragma unroll
                        for (int e = 0; e < U; ++e)
                            if (p0 + e < n) line[u * (U + 1) + e] = y[e];
                    }
                }
            }
        }
        __syncthreads();
        // ---- coalesced stores of the strip (same mapping as the fill)
        for (int i = threadIdx.x; i < items; i += EX_NT) {
            const int r0 = (i >> lk) * RB, kc = i & (kcn - 1);
            T* const o = out + static_cast<long long>(r0) * a.pitch + c0 + kc * ve;
#pragma unroll
            for (int k = 0; k < RB; ++k) {
                const int r = r0 + k;
                if (r < n) {
                    const int so = r + (r >> 3);
                    T vo[V];
                    const T* const sp = strip + static_cast<size_t>(kc * ve) * cpitch + so;
#pragma unroll
                    for (int e = 0; e < V; ++e) vo[e] = e < ve ? sp[e * cpitch] : T(0);
                    if (ve == V) st16g(o + k * a.pitch, vo);
                    else
                        for (int e = 0; e < ve; ++e) o[k * a.pitch + e] = vo[e];
                }
            }
        }
        __syncthreads();   // the strip is refilled by the next pass
    }
}

template <typename T, bool VAR, bool SEG1>
__global__ void __launch_bounds__(EX_NT) wave2d_exact_y(const __grid_constant__ ExactArgs a)
{
    extern __shared__ __align__(16) unsigned char ex_smem[];
    __shared__ ExactScratch<T> scratch;
    exact_y_half_step<T, VAR, SEG1>(a, a.n_off + 2 * (*a.d_k), ex_smem, scratch);
}

}  // namespace w2d
