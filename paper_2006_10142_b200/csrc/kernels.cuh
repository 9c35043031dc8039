// kernels.cuh -- the CUDA kernels of the ADI step (sm_100a).  See DESIGN.md for the derivation.
//
// One half-step n -> n+1 of (2.11)/(2.12) (times tau^2) is, on every grid line along
// the sweep direction, the Toeplitz tridiagonal system
//
//      -ap x_{p-1} + (gamma + 2 ap) x_p - ap x_{p+1} = r_p,          x_{-1} = x_n = 0,
//      r_p = 2 gamma wc_p - gamma wp_p + am (wp_{p-1} - 2 wp_p + wp_{p+1}) + q s_p
//
// (wp = w_{n-1}, wc = w_n).  Because c depends on t only, ap is one scalar per half-step, so the LU
// factors of the matrix are scalars too: with cp_0 = ap/beta, inv_p = 1/(beta - ap cp_{p-1}),
// cp_p = ap inv_p (-> rho, the small root of ap z^2 - beta z + ap = 0, at rate rho^{2p}),
//
//      forward   y_p = cp_p y_{p-1} + inv_p r_p          backward   x_p = y_p + cp_p x_{p+1}.
//
// Both are first-order LINEAR recurrences, so a line is cut into units of U points that are solved
// independently from a zero carry ("local" solve, one thread per unit), and the true carry is added
// afterwards:   y_{p0+e} = yloc_e + (cp_{p0} .. cp_{p0+e}) Y_in,   Y_in = y at the end of the previous unit
//                        = L_{g-1} + A_{g-1} (L_{g-2} + A_{g-2} ( ... ))        (L = last yloc, A = product of the unit's cp)
// and the same from the right for x.  A_g <= rho^U, so the carry series is cut after NBK units with
// rho^{NBK U} below the rounding unit (host-planned).  The host stores cp_p, inv_p for p < KMAX per
// half-step (exact boundary rows) and rho, 1/(beta - ap rho) for the stationary rest.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>
#include <type_traits>

#include "ptx.cuh"

namespace w2d {

// ---- per-half-step scalar table (fp64, built on the host; row n serves half-step n -> n+1) ------
constexpr int KMAX = 128;    // boundary rows with their own (cp_p, inv_p)
constexpr int NBK_MAX = 8;   // longest carry series (units)
constexpr int ROW_AM = 0, ROW_Q = 1, ROW_RHO = 2, ROW_INV = 3, ROW_C1 = 4, ROW_AP = 5, ROW_BETA = 6;
constexpr int ROW_CP = 8, ROW_INVP = 8 + KMAX, ROW_DOUBLES = 8 + 2 * KMAX;

// A piece of work: output units [ua, ub) of the 32 lines of panel `panel`; nst stages of NW units are
// streamed, starting NBK units early (carry warm-up) and ending >= NBK units late (carry look-ahead).
struct Piece {
    int panel, ua, ub, nst;
};

struct SweepArgs {
    const double* table;   // device, ROW_DOUBLES per half-step
    const int* d_k;        // device: completed time steps at graph start (NULL: 0)
    int n_off;             // half-step index = n_off + 2 * (*d_k)
    int n;                 // unknowns per line
    int nlines;            // number of lines
    int nbk;               // carry series length in units (<= NW, <= NBK_MAX)
    int kb;                // units [0, kb) use the boundary pivots of the table
    const Piece* pieces;   // device
    const int* cta_off;    // device: CTA b owns pieces [cta_off[b], cta_off[b+1])
    void* out;             // y sweep: output field (direct coalesced stores)
    long long pitch;       // row pitch in elements
    const void* src;       // compact source window, [p - sp0][line - sl0] (line fastest), or NULL
    int sl0, snl, sp0, snp;
    double g2;             // 2 gamma
};

template <typename T, int DIR, int NW, int NSTAGE>
struct PanelCfg {
    static constexpr int U = DIR == 0 ? 128 / (int)sizeof(T) : 16;   // points per unit
    static constexpr int TL = 32;                                    // lines per panel, one per lane
    static constexpr int V = 16 / (int)sizeof(T);                    // elements per 16 bytes
    // x sweep: per field NW unit tiles [32 rows][128 B] (128B-swizzled) + two edge boxes [32 rows][16 B] of wp
    // y sweep: per field one box [U*NW + 2 rows][32 columns]
    static constexpr int FIELD_BYTES = DIR == 0 ? NW * 4096 : (U * NW + 2) * TL * (int)sizeof(T);
    static constexpr int EDGE_BYTES = DIR == 0 ? 512 : 0;
    static constexpr int STAGE_BYTES = 2 * FIELD_BYTES + 2 * EDGE_BYTES;
    static constexpr int OUT_BYTES = DIR == 0 ? NW * 4096 : 0;
    static constexpr int BAR_BYTES = ((2 * NSTAGE * 8) + 15) / 16 * 16;
    static constexpr int TAB_BYTES = 2 * KMAX * (int)sizeof(T);
    static constexpr int XCH_BYTES = (4 * NW * TL + 2 * NW + 2) * (int)sizeof(T);   // Ls[2][NW][32], Hs[2][NW][32], As[2][NW]
    static constexpr int SMEM_BYTES = 1024 + NSTAGE * STAGE_BYTES + OUT_BYTES + BAR_BYTES + TAB_BYTES + XCH_BYTES;
    static constexpr int THREADS = 32 * (NW + 1);
    static_assert(FIELD_BYTES % 128 == 0, "TMA destinations must stay 128-byte aligned");
    static_assert(DIR == 0 || U * NW + 2 <= 256, "TMA box dimension limit");
};

// Read this lane's line of one x-sweep unit tile [32 rows][128 B] into registers; the tile is
// 128B-swizzled by TMA: 16-byte chunk c of row t sits at chunk c ^ (t & 7)  (bank-conflict-free).
template <typename T>
__device__ __forceinline__ void load_unit_x(const unsigned char* tile, int lane, T (&v)[128 / sizeof(T)])
{
    const unsigned char* row = tile + lane * 128;
    const int sw = (lane & 7) << 4;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        if constexpr (sizeof(T) == 8) {
            const double2 t = *reinterpret_cast<const double2*>(row + ((c << 4) ^ sw));
            v[2 * c] = t.x;
            v[2 * c + 1] = t.y;
        } else {
            const float4 t = *reinterpret_cast<const float4*>(row + ((c << 4) ^ sw));
            v[4 * c] = t.x;
            v[4 * c + 1] = t.y;
            v[4 * c + 2] = t.z;
            v[4 * c + 3] = t.w;
        }
    }
}
// first / last element of this lane's row of an x-sweep unit tile
template <typename T>
__device__ __forceinline__ T tile_first_x(const unsigned char* tile, int lane)
{
    return *reinterpret_cast<const T*>(tile + lane * 128 + ((lane & 7) << 4));
}
template <typename T>
__device__ __forceinline__ T tile_last_x(const unsigned char* tile, int lane)
{
    return *reinterpret_cast<const T*>(tile + lane * 128 + ((7 ^ (lane & 7)) << 4) + 16 - sizeof(T));
}

__device__ __forceinline__ void named_bar_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// ---------------------------------------------------------------------------------------------------
// Panel sweep: RHS assembly (A1/A3) fused with the line solve (A2/A4), SURVEY.md 8a.
//   grid  = persistent CTAs (SM count x CTAs/SM); CTA b walks its host-planned pieces.
//   block = NW consumer warps + 1 producer warp (one lane issues TMA).  Per stage, consumer warp w
//           owns unit g = gbase + s*NW + w of the panel's 32 lines, lane = line.
//   stage:  smem -> registers, release the slot; RHS + local forward; publish L, A; bar;
//           carry-in, correct y, local backward; publish head; bar;
//           finish the unit of the PREVIOUS stage (its look-ahead heads are now known) and store it.
// ---------------------------------------------------------------------------------------------------
template <typename T, int DIR, int NW, int NSTAGE>
__global__ void __launch_bounds__(32 * (NW + 1), 1)
wave2d_sweep_panel(const __grid_constant__ CUtensorMap tm_prev, const __grid_constant__ CUtensorMap tm_cur,
                   const __grid_constant__ CUtensorMap tm_out, const __grid_constant__ CUtensorMap tm_edge,
                   const SweepArgs a)
{
    using K = PanelCfg<T, DIR, NW, NSTAGE>;
    constexpr int U = K::U, TL = K::TL, V = K::V;

    extern __shared__ unsigned char smem_raw[];
    const uint32_t raw32 = smem_u32(smem_raw);
    const uint32_t pad = ((raw32 + 1023u) & ~1023u) - raw32;
    unsigned char* sm = smem_raw + pad;   // 1024-byte aligned: the 128B-swizzle atom
    const uint32_t sm32 = raw32 + pad;
    unsigned char* sm_out = sm + NSTAGE * K::STAGE_BYTES;
    const uint32_t bar32 = sm32 + NSTAGE * K::STAGE_BYTES + K::OUT_BYTES;   // full[NSTAGE], empty[NSTAGE]
    T* s_cp = reinterpret_cast<T*>(sm + NSTAGE * K::STAGE_BYTES + K::OUT_BYTES + K::BAR_BYTES);
    T* s_inv = s_cp + KMAX;
    T* s_L = s_inv + KMAX;            // [2][NW][32]  last local y of a unit
    T* s_H = s_L + 2 * NW * TL;       // [2][NW][32]  first local x of a unit
    T* s_A = s_H + 2 * NW * TL;       // [2][NW]      product of the unit's cp

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nh = a.n_off + (a.d_k ? 2 * (*a.d_k) : 0);
    const double* row = a.table + static_cast<size_t>(nh) * ROW_DOUBLES;

    for (int i = threadIdx.x; i < KMAX; i += K::THREADS) {
        s_cp[i] = static_cast<T>(row[ROW_CP + i]);
        s_inv[i] = static_cast<T>(row[ROW_INVP + i]);
    }
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NSTAGE; ++s) {
            mbar_init(bar32 + 8 * s, 1);
            mbar_init(bar32 + 8 * (NSTAGE + s), NW);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int pc_begin = a.cta_off[blockIdx.x], pc_end = a.cta_off[blockIdx.x + 1];

    if (warp == NW) {   // ---------------- producer: one lane feeds the stage ring by TMA
        if (lane == 0) {
            tma_prefetch_desc(&tm_prev);
            tma_prefetch_desc(&tm_cur);
            int it = 0;
            for (int pi = pc_begin; pi < pc_end; ++pi) {
                const Piece pc = a.pieces[pi];
                const int line0 = pc.panel * TL;
                const int gbase = max(pc.ua - a.nbk, 0);
                for (int s = 0; s < pc.nst; ++s, ++it) {
                    const int slot = it % NSTAGE;
                    if (it >= NSTAGE) mbar_wait(bar32 + 8 * (NSTAGE + slot), ((it / NSTAGE) - 1) & 1);
                    const uint32_t full = bar32 + 8 * slot;
                    mbar_arrive_expect_tx(full, K::STAGE_BYTES);
                    const uint32_t dst = sm32 + slot * K::STAGE_BYTES;
                    const int g0 = gbase + s * NW;
                    if constexpr (DIR == 0) {
#pragma unroll
                        for (int w = 0; w < NW; ++w) {
                            tma_load_2d(dst + w * 4096, &tm_prev, (g0 + w) * U, line0, full);
                            tma_load_2d(dst + K::FIELD_BYTES + w * 4096, &tm_cur, (g0 + w) * U, line0, full);
                        }
                        tma_load_2d(dst + 2 * K::FIELD_BYTES, &tm_edge, g0 * U - V, line0, full);
                        tma_load_2d(dst + 2 * K::FIELD_BYTES + K::EDGE_BYTES, &tm_edge, (g0 + NW) * U, line0, full);
                    } else {
                        tma_load_2d(dst, &tm_prev, line0, g0 * U - 1, full);
                        tma_load_2d(dst + K::FIELD_BYTES, &tm_cur, line0, g0 * U - 1, full);
                    }
                }
            }
        }
        return;
    }

    // -------------------- consumers
    const T am = static_cast<T>(row[ROW_AM]), q = static_cast<T>(row[ROW_Q]), rho = static_cast<T>(row[ROW_RHO]);
    const T inv = static_cast<T>(row[ROW_INV]), c1 = static_cast<T>(row[ROW_C1]), g2 = static_cast<T>(a.g2);
    const int n = a.n, nbk = a.nbk;
    T pw[U];   // pw[e] = rho^(e+1)
    pw[0] = rho;
#pragma unroll
    for (int e = 1; e < U; ++e) pw[e] = pw[e - 1] * rho;
    auto cp_at = [&](int p) -> T { return p < KMAX ? s_cp[p] : rho; };
    auto inv_at = [&](int p) -> T { return p < KMAX ? s_inv[p] : inv; };

    T pend[U];
#pragma unroll
    for (int e = 0; e < U; ++e) pend[e] = T(0);
    int it = 0;

    for (int pi = pc_begin; pi < pc_end; ++pi) {
        const Piece pc = a.pieces[pi];
        const int line0 = pc.panel * TL, line = line0 + lane;
        const int gbase = max(pc.ua - nbk, 0);
        const bool src_tile = a.src != nullptr && line0 < a.sl0 + a.snl && line0 + TL > a.sl0;
        const bool src_line = line >= a.sl0 && line < a.sl0 + a.snl;
        const T* srcp = reinterpret_cast<const T*>(a.src) + (line - a.sl0);

        named_bar_sync(1, NW * 32);   // the previous piece is completely finished
        s_L[(NW + warp) * TL + lane] = T(0);   // "stage -1": zero carries
        if (lane == 0) s_A[NW + warp] = T(0);

        for (int s = 0; s <= pc.nst; ++s) {
            const int buf = s & 1;
            const int g = gbase + s * NW + warp, p0 = g * U;
            const bool act = s < pc.nst;
            bool fast = false;
            T xl[U];
#pragma unroll
            for (int e = 0; e < U; ++e) xl[e] = T(0);

            if (act) {
                const int slot = it % NSTAGE;
                mbar_wait(bar32 + 8 * slot, (it / NSTAGE) & 1);
                ++it;
                const unsigned char* st = sm + slot * K::STAGE_BYTES;
                T wp[U], wc[U], wl, wr;
                if constexpr (DIR == 0) {
                    const unsigned char* tp = st + warp * 4096;
                    load_unit_x<T>(tp, lane, wp);
                    load_unit_x<T>(st + K::FIELD_BYTES + warp * 4096, lane, wc);
                    wl = warp == 0 ? reinterpret_cast<const T*>(st + 2 * K::FIELD_BYTES)[lane * V + V - 1]
                                   : tile_last_x<T>(tp - 4096, lane);
                    wr = warp == NW - 1 ? reinterpret_cast<const T*>(st + 2 * K::FIELD_BYTES + K::EDGE_BYTES)[lane * V]
                                        : tile_first_x<T>(tp + 4096, lane);
                } else {
                    const T* cpv = reinterpret_cast<const T*>(st) + (warp * U) * TL + lane;
                    const T* ccv = reinterpret_cast<const T*>(st + K::FIELD_BYTES) + (warp * U + 1) * TL + lane;
                    wl = cpv[0];
#pragma unroll
                    for (int e = 0; e < U; ++e) wp[e] = cpv[(e + 1) * TL];
                    wr = cpv[(U + 1) * TL];
#pragma unroll
                    for (int e = 0; e < U; ++e) wc[e] = ccv[e * TL];
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar32 + 8 * (NSTAGE + slot));   // data is in registers: release the slot

                const bool src_k = src_tile && p0 < a.sp0 + a.snp && p0 + U > a.sp0;
                fast = g >= a.kb && p0 + U <= n && !src_k;
                T Aval;
                if (fast) {   // stationary pivots: y_e = rho y_{e-1} + inv r_e from y_{-1} = 0
                    T fy = T(0);
#pragma unroll
                    for (int e = 0; e < U; ++e) {
                        const T left = e == 0 ? wl : wp[e - 1];
                        const T right = e == U - 1 ? wr : wp[e + 1];
                        const T r = fma(g2, wc[e], fma(am, left + right, c1 * wp[e]));
                        fy = fma(rho, fy, r * inv);
                        xl[e] = fy;
                    }
                    Aval = pw[U - 1];
                } else {
                    const bool src_unit = src_k && src_line;
                    T fy = T(0), prod = T(1);
#pragma unroll
                    for (int e = 0; e < U; ++e) {
                        const int p = p0 + e;
                        const T left = e == 0 ? wl : wp[e - 1];
                        const T right = e == U - 1 ? wr : wp[e + 1];
                        T r = fma(g2, wc[e], fma(am, left + right, c1 * wp[e]));
                        if (src_unit && p >= a.sp0 && p < a.sp0 + a.snp)
                            r = fma(q, srcp[static_cast<size_t>(p - a.sp0) * a.snl], r);
                        const T cpe = cp_at(p);
                        fy = fma(cpe, fy, r * inv_at(p));
                        if (p >= n) fy = T(0);
                        prod *= cpe;
                        xl[e] = fy;
                    }
                    Aval = prod;
                }
                s_L[(buf * NW + warp) * TL + lane] = xl[U - 1];
                if (lane == 0) s_A[buf * NW + warp] = Aval;
            }
            named_bar_sync(1, NW * 32);

            if (act) {
                T Yin = T(0);   // y at the end of unit g-1
                for (int j = nbk; j >= 1; --j) {
                    int idx = warp - j, b = buf;
                    if (idx < 0) { idx += NW; b ^= 1; }
                    Yin = fma(s_A[b * NW + idx], Yin, s_L[(b * NW + idx) * TL + lane]);
                }
                if (fast) {
#pragma unroll
                    for (int e = 0; e < U; ++e) xl[e] = fma(pw[e], Yin, xl[e]);
#pragma unroll
                    for (int e = U - 2; e >= 0; --e) xl[e] = fma(rho, xl[e + 1], xl[e]);
                } else {
                    T c = Yin;
#pragma unroll
                    for (int e = 0; e < U; ++e) {
                        c *= cp_at(p0 + e);
                        xl[e] = p0 + e < n ? xl[e] + c : T(0);
                    }
#pragma unroll
                    for (int e = U - 2; e >= 0; --e) xl[e] = fma(cp_at(p0 + e), xl[e + 1], xl[e]);
                }
            }
            s_H[(buf * NW + warp) * TL + lane] = xl[0];   // 0 in the flush stage
            named_bar_sync(1, NW * 32);

            if (s > 0) {   // finish the unit of stage s-1: gp = g - NW, local x in pend[]
                const int gp = g - NW, pp0 = gp * U;
                T Xin = T(0);   // x at the start of unit gp+1
                for (int j = nbk; j >= 1; --j) {
                    int idx = warp + j, b = buf ^ 1;
                    if (idx >= NW) { idx -= NW; b ^= 1; }
                    Xin = fma(s_A[b * NW + idx], Xin, s_H[(b * NW + idx) * TL + lane]);
                }
                if (gp >= pc.ua && gp < pc.ub) {   // warp-uniform
                    if (gp >= a.kb && pp0 + U <= n) {
#pragma unroll
                        for (int e = 0; e < U; ++e) pend[e] = fma(pw[U - 1 - e], Xin, pend[e]);
                    } else {
                        T c = Xin;
#pragma unroll
                        for (int e = U - 1; e >= 0; --e) {
                            c *= cp_at(pp0 + e);
                            pend[e] += c;
                        }
                    }
                    if constexpr (DIR == 0) {
                        unsigned char* ot = sm_out + warp * 4096;
                        if (lane == 0) tma_wait_read<0>();   // the previous store of this warp has read the tile
                        __syncwarp();
                        unsigned char* orow = ot + lane * 128;
                        const int sw = (lane & 7) << 4;
#pragma unroll
                        for (int c = 0; c < 8; ++c) {
                            if constexpr (sizeof(T) == 8)
                                *reinterpret_cast<double2*>(orow + ((c << 4) ^ sw)) = make_double2(pend[2 * c], pend[2 * c + 1]);
                            else
                                *reinterpret_cast<float4*>(orow + ((c << 4) ^ sw)) =
                                    make_float4(pend[4 * c], pend[4 * c + 1], pend[4 * c + 2], pend[4 * c + 3]);
                        }
                        fence_async_smem();
                        __syncwarp();
                        if (lane == 0) {
                            tma_store_2d(&tm_out, pp0, line0, smem_u32(ot));
                            tma_commit();
                        }
                    } else {
                        if (line < a.nlines) {
                            T* o = reinterpret_cast<T*>(a.out) + static_cast<long long>(pp0) * a.pitch + line;
#pragma unroll
                            for (int e = 0; e < U; ++e)
                                if (pp0 + e < n) o[static_cast<long long>(e) * a.pitch] = pend[e];
                        }
                    }
                }
            }
#pragma unroll
            for (int e = 0; e < U; ++e) pend[e] = xl[e];
        }
    }
    if constexpr (DIR == 0) {
        if (lane == 0) tma_wait_read<0>();
    }
}

// ---------------------------------------------------------------------------------------------------
// Exact path (any tau/h): plain Thomas elimination with the half-step's own pivots, one thread per
// line, two passes through HBM (forward writes y into `out`, backward turns it into x in place).
// Used when rho^H cannot be made negligible within the look-ahead the streamed kernel supports, or
// on request (WAVE2D_SOLVER_EXACT).  DIR 1 is coalesced; DIR 0 walks rows and is slow but correct.
// ---------------------------------------------------------------------------------------------------
// cpv[p], ivv[p], p < n: one thread block; thread 0 runs the pivot recurrence until it is stationary.
__global__ void wave2d_exact_pivots(const double* table, const int* d_k, int n_off, int n, double* cpv, double* ivv)
{
    __shared__ int s_conv;
    const int nh = n_off + (d_k ? 2 * (*d_k) : 0);
    const double* row = table + static_cast<size_t>(nh) * ROW_DOUBLES;
    const double ap = row[ROW_AP], beta = row[ROW_BETA];
    if (threadIdx.x == 0) {
        double cp = 0.0;
        int p = 0;
        for (; p < n; ++p) {
            const double iv = 1.0 / (beta - ap * cp);
            const double cn = ap * iv;
            cpv[p] = cn;
            ivv[p] = iv;
            if (cn == cp) { ++p; break; }
            cp = cn;
        }
        s_conv = p;
    }
    __syncthreads();
    const int pc = s_conv;
    if (pc < n) {
        const double cp = cpv[pc - 1], iv = ivv[pc - 1];
        for (int p = pc + threadIdx.x; p < n; p += blockDim.x) {
            cpv[p] = cp;
            ivv[p] = iv;
        }
    }
}

template <typename T, int DIR>
__global__ void wave2d_exact_forward(const T* __restrict__ wprev, const T* __restrict__ wcur, T* __restrict__ out,
                                     const double* table, const int* d_k, int n_off, int n, int nlines,
                                     long long pitch, const double* __restrict__ cpv, const double* __restrict__ ivv,
                                     const T* __restrict__ src, int sl0, int snl, int sp0, int snp, double g2d)
{
    const int line = blockIdx.x * blockDim.x + threadIdx.x;
    if (line >= nlines) return;
    const int nh = n_off + (d_k ? 2 * (*d_k) : 0);
    const double* row = table + static_cast<size_t>(nh) * ROW_DOUBLES;
    const T am = static_cast<T>(row[ROW_AM]), q = static_cast<T>(row[ROW_Q]), c1 = static_cast<T>(row[ROW_C1]);
    const T g2 = static_cast<T>(g2d);
    const long long ls = DIR == 0 ? pitch : 1, ps = DIR == 0 ? 1 : pitch;   // strides between lines / along the line
    const T* wp = wprev + line * ls;
    const T* wc = wcur + line * ls;
    T* o = out + line * ls;
    const bool src_line = src != nullptr && line >= sl0 && line < sl0 + snl;
    T left = T(0), mid = n > 0 ? wp[0] : T(0), fy = T(0);
    for (int p = 0; p < n; ++p) {
        const T right = p + 1 < n ? wp[(p + 1) * ps] : T(0);
        T r = fma(g2, wc[p * ps], fma(am, left + right, c1 * mid));
        if (src_line && p >= sp0 && p < sp0 + snp) r = fma(q, src[static_cast<size_t>(p - sp0) * snl + (line - sl0)], r);
        fy = fma(static_cast<T>(cpv[p]), fy, r * static_cast<T>(ivv[p]));
        o[p * ps] = fy;
        left = mid;
        mid = right;
    }
}

template <typename T, int DIR>
__global__ void wave2d_exact_backward(T* __restrict__ out, int n, int nlines, long long pitch,
                                      const double* __restrict__ cpv)
{
    const int line = blockIdx.x * blockDim.x + threadIdx.x;
    if (line >= nlines) return;
    const long long ls = DIR == 0 ? pitch : 1, ps = DIR == 0 ? 1 : pitch;
    T* o = out + line * ls;
    T x = T(0);
    for (int p = n - 1; p >= 0; --p) {
        x = fma(static_cast<T>(cpv[p]), x, o[p * ps]);
        o[p * ps] = x;
    }
}

// ---- A-init (PAPER.md:68-69 (2.9)): w_{-1} = phi - (tau/2) psi -----------------
template <typename T>
__global__ void wave2d_init_prev(T* __restrict__ prev, const T* __restrict__ phi, const T* __restrict__ psi,
                                 int n1, int n2, long long pitch, double half_tau)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= n1 || j >= n2) return;
    const long long o = j * pitch + i;
    prev[o] = psi ? static_cast<T>(phi[o] - static_cast<T>(half_tau) * psi[o]) : phi[o];
}

// dst[p][l] = src[l][p] for a small window (compact source, transposed copy for the x sweep)
template <typename T>
__global__ void wave2d_transpose_small(T* __restrict__ dst, const T* __restrict__ src, int rows, int cols)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x, r = blockIdx.y;
    if (c < cols && r < rows) dst[static_cast<size_t>(c) * rows + r] = src[static_cast<size_t>(r) * cols + c];
}

__global__ void wave2d_bump_counter(int* d_k, int by) { *d_k += by; }

}  // namespace w2d
