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
// Both are first-order recurrences with memory rho^k, so a line can be cut into chunks that each
// start H points early (forward) and look H points ahead (backward) with rho^H below the rounding
// unit.  The host stores cp_p, inv_p for p < K per half-step (exact boundary rows) and rho, 1/(beta-ap rho).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>
#include <type_traits>

#include "ptx.cuh"

namespace w2d {

// ---- per-half-step scalar table (fp64, built on the host; row n serves half-step n -> n+1) ------
constexpr int KMAX = 64;   // boundary rows with their own (cp_p, inv_p)
constexpr int ROW_AM = 0, ROW_Q = 1, ROW_RHO = 2, ROW_INV = 3, ROW_C1 = 4, ROW_AP = 5, ROW_BETA = 6;
constexpr int ROW_CP = 8, ROW_INVP = 8 + KMAX, ROW_DOUBLES = 8 + 2 * KMAX;

struct SweepArgs {
    const double* table;   // device, ROW_DOUBLES per half-step
    const int* d_k;        // device: completed time steps at graph start (NULL: 0)
    int n_off;             // half-step index = n_off + 2 * (*d_k)
    int n;                 // unknowns per line
    int nlines;            // number of lines
    int ntiles;            // ceil(nlines / TL)
    int upc;               // units per chunk
    int total_units;       // ceil(n / U)
    void* out;             // y sweep: output field (direct coalesced stores)
    long long pitch;       // row pitch in elements
    const void* src;       // compact source window, [p - sp0][line - sl0] (line fastest), or NULL
    int sl0, snl, sp0, snp;
    double g2;             // 2 gamma
};

template <typename T, int DIR, int NB, int NW, int XB, int NSTAGE>
struct StreamCfg {
    static constexpr int U = 128 / sizeof(T);          // points per unit (one 128-byte swizzle row)
    static constexpr int TL = 32 * NW;                 // lines per CTA, one per consumer thread
    static constexpr int UNIT_BYTES = TL * 128;        // one unit of one field
    static constexpr int STAGE_BYTES = 2 * XB * UNIT_BYTES;
    static constexpr int OUT_BYTES = DIR == 0 ? NW * 2 * 32 * 128 : 0;
    static constexpr int BAR_BYTES = ((2 * NSTAGE * 8) + 15) / 16 * 16;
    static constexpr int TAB_BYTES = 2 * KMAX * sizeof(T);
    static constexpr int SMEM_BYTES = 1024 + NSTAGE * STAGE_BYTES + OUT_BYTES + BAR_BYTES + TAB_BYTES;
    static constexpr int THREADS = 32 * (NW + 1);
};

// Read this thread's line of one unit tile into registers.
//   DIR 0 (x sweep): tile = [TL rows][128 B], 128B-swizzled by TMA: 16-byte chunk c of row t sits at chunk c ^ (t & 7).
//   DIR 1 (y sweep): tile = [U rows][TL columns], dense.
template <typename T, int DIR, int TL>
__device__ __forceinline__ void load_unit(const unsigned char* tile, int tid, T (&v)[128 / sizeof(T)])
{
    constexpr int U = 128 / sizeof(T);
    if constexpr (DIR == 0) {
        const unsigned char* row = tile + tid * 128;
        const int sw = (tid & 7) << 4;
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
    } else {
        const T* col = reinterpret_cast<const T*>(tile) + tid;
#pragma unroll
        for (int e = 0; e < U; ++e) v[e] = col[e * TL];
    }
}

template <typename T, int DIR, int TL>
__device__ __forceinline__ T peek_first(const unsigned char* tile, int tid)
{
    if constexpr (DIR == 0)
        return *reinterpret_cast<const T*>(tile + tid * 128 + ((tid & 7) << 4));
    else
        return reinterpret_cast<const T*>(tile)[tid];
}

// ---------------------------------------------------------------------------------------------------
// Streamed sweep: RHS assembly (A1/A3) fused with the line solve (A2/A4), SURVEY.md 8a.
//   grid  = ntiles * nchunks CTAs; CTA (tile, chunk) owns lines [tile*TL, +TL) and output units
//           [chunk*upc, +upc) of every one of them; it streams units [first - NB, last + NB].
//   block = NW consumer warps (one thread per line) + 1 producer warp (one lane issues TMA).
// ---------------------------------------------------------------------------------------------------
template <typename T, int DIR, int NB, int NW, int XB, int NSTAGE>
__global__ void __launch_bounds__(32 * (NW + 1))
wave2d_sweep_stream(const __grid_constant__ CUtensorMap tm_prev, const __grid_constant__ CUtensorMap tm_cur,
                    const __grid_constant__ CUtensorMap tm_out, const SweepArgs a)
{
    using K = StreamCfg<T, DIR, NB, NW, XB, NSTAGE>;
    constexpr int U = K::U, TL = K::TL, RING = (NB + 1) * U;
    static_assert(NB * U <= KMAX, "boundary table too short");

    extern __shared__ unsigned char smem_raw[];
    const uint32_t raw32 = smem_u32(smem_raw);
    const uint32_t pad = ((raw32 + 1023u) & ~1023u) - raw32;
    unsigned char* sm = smem_raw + pad;   // 1024-byte aligned: the 128B-swizzle atom
    const uint32_t sm32 = raw32 + pad;
    unsigned char* sm_out = sm + NSTAGE * K::STAGE_BYTES;
    const uint32_t bar32 = sm32 + NSTAGE * K::STAGE_BYTES + K::OUT_BYTES;   // full[NSTAGE], empty[NSTAGE]
    T* s_cp = reinterpret_cast<T*>(sm + NSTAGE * K::STAGE_BYTES + K::OUT_BYTES + K::BAR_BYTES);
    T* s_inv = s_cp + KMAX;

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

    const int tile = blockIdx.x % a.ntiles, chunk = blockIdx.x / a.ntiles;
    const int line0 = tile * TL;
    const int uo0 = chunk * a.upc;                                         // output units [uo0, uo1)
    const int uo1 = min(uo0 + a.upc, a.total_units);
    const int ub = max(uo0 - NB, 0);                                       // first streamed unit
    const int ue_want = (uo1 == a.total_units ? a.total_units : uo1) + NB; // lookahead / flush units
    const int ns = (ue_want - ub + XB - 1) / XB;                           // stages

    if (warp == NW) {   // ---------------- producer: one lane feeds the stage ring by TMA
        if (lane == 0) {
            tma_prefetch_desc(&tm_prev);
            tma_prefetch_desc(&tm_cur);
            for (int s = 0; s < ns; ++s) {
                const int slot = s % NSTAGE;
                if (s >= NSTAGE) mbar_wait(bar32 + 8 * (NSTAGE + slot), ((s / NSTAGE) - 1) & 1);
                const uint32_t full = bar32 + 8 * slot;
                mbar_arrive_expect_tx(full, K::STAGE_BYTES);
                const uint32_t dst = sm32 + slot * K::STAGE_BYTES;
                const int u0 = ub + s * XB;
                if constexpr (DIR == 0) {
#pragma unroll
                    for (int xb = 0; xb < XB; ++xb) {
                        tma_load_2d(dst + xb * K::UNIT_BYTES, &tm_prev, (u0 + xb) * U, line0, full);
                        tma_load_2d(dst + (XB + xb) * K::UNIT_BYTES, &tm_cur, (u0 + xb) * U, line0, full);
                    }
                } else {
                    tma_load_2d(dst, &tm_prev, line0, u0 * U, full);
                    tma_load_2d(dst + XB * K::UNIT_BYTES, &tm_cur, line0, u0 * U, full);
                }
            }
        }
        return;
    }

    // -------------------- consumers: thread tid owns line line0 + tid
    const int tid = threadIdx.x;
    const int line = line0 + tid;
    const T am = static_cast<T>(row[ROW_AM]), q = static_cast<T>(row[ROW_Q]), rho = static_cast<T>(row[ROW_RHO]);
    const T inv = static_cast<T>(row[ROW_INV]), c1 = static_cast<T>(row[ROW_C1]), g2 = static_cast<T>(a.g2);
    const int n = a.n;
    const bool src_tile = a.src != nullptr && line0 < a.sl0 + a.snl && line0 + TL > a.sl0;
    const bool src_line = line >= a.sl0 && line < a.sl0 + a.snl;
    const T* srcp = reinterpret_cast<const T*>(a.src) + (line - a.sl0);

    T ring[RING];   // y of the last NB+1 units, oldest first
#pragma unroll
    for (int e = 0; e < RING; ++e) ring[e] = T(0);
    T fy = T(0), wp_last = T(0);
    int ob = 0;

    auto unit = [&](auto gen_c, const unsigned char* tprev, const unsigned char* tcur, T peek, int k) {
        constexpr bool GEN = decltype(gen_c)::value;
        T wp[U], wc[U];
        load_unit<T, DIR, TL>(tprev, tid, wp);
        load_unit<T, DIR, TL>(tcur, tid, wc);
#pragma unroll
        for (int e = 0; e < NB * U; ++e) ring[e] = ring[e + U];
        const int p0 = k * U;
        const bool tab_new = GEN && k < NB;
        const bool src_unit = GEN && src_tile && src_line;
        // ---- RHS (A1/A3) and forward elimination
#pragma unroll
        for (int e = 0; e < U; ++e) {
            const T left = e == 0 ? wp_last : wp[e - 1];
            const T right = e == U - 1 ? peek : wp[e + 1];
            T r = fma(g2, wc[e], fma(am, left + right, c1 * wp[e]));
            T cpe = rho, ive = inv;
            if constexpr (GEN) {
                const int p = p0 + e;
                if (src_unit && p >= a.sp0 && p < a.sp0 + a.snp)
                    r = fma(q, srcp[static_cast<size_t>(p - a.sp0) * a.snl], r);
                if (tab_new) {
                    cpe = s_cp[p];
                    ive = s_inv[p];
                }
            }
            fy = fma(cpe, fy, r * ive);
            T v = fy;
            if constexpr (GEN) {
                if (p0 + e >= n) v = T(0);
            }
            ring[NB * U + e] = v;
        }
        wp_last = wp[U - 1];
        // ---- back substitution: NB units of look-ahead, then the unit that is NB behind
        T x = T(0);
#pragma unroll
        for (int e = RING - 1; e >= U; --e) {
            T cpe = rho;
            if constexpr (GEN) {
                const int p = (k - NB) * U + e;
                if (p >= 0 && p < NB * U) cpe = s_cp[p];
            }
            x = fma(cpe, x, ring[e]);
        }
        const int ko = k - NB;
        if (ko >= uo0 && ko < uo1) {
            if constexpr (DIR == 0) {
                unsigned char* ot = sm_out + (warp * 2 + ob) * 4096;
                if (lane == 0) tma_wait_read<1>();
                __syncwarp();
                unsigned char* orow = ot + lane * 128;
                const int sw = (lane & 7) << 4;
                constexpr int V = 16 / sizeof(T);
#pragma unroll
                for (int c = 7; c >= 0; --c) {
                    T xo[V];
#pragma unroll
                    for (int i = V - 1; i >= 0; --i) {
                        T cpe = rho;
                        if constexpr (GEN) {
                            const int p = ko * U + c * V + i;
                            if (p < NB * U) cpe = s_cp[p];
                        }
                        x = fma(cpe, x, ring[c * V + i]);
                        xo[i] = x;
                    }
                    if constexpr (sizeof(T) == 8)
                        *reinterpret_cast<double2*>(orow + ((c << 4) ^ sw)) = make_double2(xo[0], xo[1]);
                    else
                        *reinterpret_cast<float4*>(orow + ((c << 4) ^ sw)) = make_float4(xo[0], xo[1], xo[2], xo[3]);
                }
                fence_async_smem();
                __syncwarp();
                if (lane == 0) {
                    tma_store_2d(&tm_out, ko * U, line0 + warp * 32, smem_u32(ot));
                    tma_commit();
                }
                ob ^= 1;
            } else {
                T* o = reinterpret_cast<T*>(a.out) + static_cast<long long>(ko * U) * a.pitch + line;
                const bool line_ok = line < a.nlines;
#pragma unroll
                for (int e = U - 1; e >= 0; --e) {
                    T cpe = rho;
                    if constexpr (GEN) {
                        const int p = ko * U + e;
                        if (p < NB * U) cpe = s_cp[p];
                    }
                    x = fma(cpe, x, ring[e]);
                    bool ok = line_ok;
                    if constexpr (GEN) ok = ok && (ko * U + e < n);
                    if (ok) o[static_cast<long long>(e) * a.pitch] = x;
                }
            }
        }
    };

    mbar_wait(bar32, 0);
    for (int s = 0; s < ns; ++s) {
        const int slot = s % NSTAGE;
        const unsigned char* st = sm + slot * K::STAGE_BYTES;
        const bool has_next = s + 1 < ns;
        const int nslot = (s + 1) % NSTAGE;
#pragma unroll
        for (int xb = 0; xb < XB; ++xb) {
            const int k = ub + s * XB + xb;
            T peek = T(0);
            if (xb + 1 < XB) {
                peek = peek_first<T, DIR, TL>(st + (xb + 1) * K::UNIT_BYTES, tid);
            } else if (has_next) {
                mbar_wait(bar32 + 8 * nslot, ((s + 1) / NSTAGE) & 1);   // the next stage is also this loop's next wait
                peek = peek_first<T, DIR, TL>(sm + nslot * K::STAGE_BYTES, tid);
            }
            const bool src_k = src_tile && k * U < a.sp0 + a.snp && (k + 1) * U > a.sp0;
            const bool fast = k >= 2 * NB && (k + 1) * U <= n && !src_k;
            if (fast)
                unit(std::false_type{}, st + xb * K::UNIT_BYTES, st + (XB + xb) * K::UNIT_BYTES, peek, k);
            else
                unit(std::true_type{}, st + xb * K::UNIT_BYTES, st + (XB + xb) * K::UNIT_BYTES, peek, k);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar32 + 8 * (NSTAGE + slot));
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
