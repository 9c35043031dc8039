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

// ---- two fp32 lines in one lane --------------------------------------------------------------------
// The fp32 y sweep runs the kernel below with T = vec2f: a lane owns two adjacent grid columns (8 bytes), so
// a panel is 64 columns and its rows are 256 contiguous bytes like in the fp64 y sweep.  All arithmetic is
// element-wise; the scalar table entries are broadcast to both elements.
struct __align__(8) vec2f {
    float x, y;
    vec2f() = default;
    __device__ __forceinline__ vec2f(float a, float b) : x(a), y(b) {}
    __device__ __forceinline__ vec2f(int a) : x(static_cast<float>(a)), y(static_cast<float>(a)) {}
    __device__ __forceinline__ explicit vec2f(double a) : x(static_cast<float>(a)), y(static_cast<float>(a)) {}
    __device__ __forceinline__ vec2f& operator+=(const vec2f& b);
    __device__ __forceinline__ vec2f& operator*=(const vec2f& b);
};
// Blackwell's packed fp32 pipe: one FFMA2 / FMUL2 / FADD2 works on both elements of a 64-bit register pair
// (fma.rn.f32x2 etc., sm_100+), rounding each element exactly like the scalar instruction.
__device__ __forceinline__ unsigned long long pack2(const vec2f& a)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y));
    return r;
}
__device__ __forceinline__ vec2f unpack2(unsigned long long r)
{
    vec2f a;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a.x), "=f"(a.y) : "l"(r));
    return a;
}
__device__ __forceinline__ vec2f operator+(const vec2f& a, const vec2f& b)
{
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pack2(a)), "l"(pack2(b)));
    return unpack2(r);
}
__device__ __forceinline__ vec2f operator*(const vec2f& a, const vec2f& b)
{
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pack2(a)), "l"(pack2(b)));
    return unpack2(r);
}
__device__ __forceinline__ vec2f fmaT(const vec2f& a, const vec2f& b, const vec2f& c)
{
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(pack2(a)), "l"(pack2(b)), "l"(pack2(c)));
    return unpack2(r);
}
__device__ __forceinline__ vec2f& vec2f::operator+=(const vec2f& b) { *this = *this + b; return *this; }
__device__ __forceinline__ vec2f& vec2f::operator*=(const vec2f& b) { *this = *this * b; return *this; }
__device__ __forceinline__ double fmaT(double a, double b, double c) { return ::fma(a, b, c); }
__device__ __forceinline__ float fmaT(float a, float b, float c) { return ::fmaf(a, b, c); }

// ---- per-half-step scalar table (fp64, built on the host; row n serves half-step n -> n+1) ------
constexpr int KMAX = 256;    // boundary rows with their own (cp_p, inv_p); >= the longest line of the small-grid kernel
constexpr int NBK_MAX = 8;   // longest carry series (units)
constexpr int ROW_AM = 0, ROW_Q = 1, ROW_RHO = 2, ROW_INV = 3, ROW_C1 = 4, ROW_AP = 5, ROW_BETA = 6, ROW_LNR = 7;
constexpr int ROW_CP = 8, ROW_INVP = 8 + KMAX, ROW_DOUBLES = 8 + 2 * KMAX;

// A piece of work: output units [ua, ub) of the 32 lines of panel `panel`; nst stages of NW units are
// streamed, starting NBK units early (carry warm-up) and ending >= NBK units late (carry look-ahead).
struct Piece {
    int panel, ua, ub, nst;
    int safe;   // 1: touches only lines the previous sweep finished in its static part (may start before it ends)
};

// Buffer roles of sweep nh (two sweeps per solve), computed on the device from the step counter so that one
// captured graph serves every phase of the ring (A6).
//   ring 3 (scheme 0): reads w_{n-1} = B[n % 3], w_n = B[(n+1) % 3], writes w_{n+1} = B[(n+2) % 3].
//   ring 4 (scheme 1): t = nh / 2 solves done: U^k = B[t % 4], V^{k-1} = B[(t+1) % 4], V^k = B[(t+2) % 4];
//             x sweep: "prev" = V^{k-1}, "cur" = U^k, writes V^{k+1} into B[(t+3) % 4];
//             y sweep: right-hand side V^{k+1} (as "prev" and "cur"), writes U^{k+1} over V^{k-1}.
struct Roles {
    int prev, cur, out;
};
__host__ __device__ __forceinline__ Roles roles_of(int nh, int ring)
{
    if (ring == 3) return Roles{nh % 3, (nh + 1) % 3, (nh + 2) % 3};
    const int t = nh >> 1;
    if ((nh & 1) == 0) return Roles{(t + 1) & 3, t & 3, (t + 3) & 3};
    return Roles{(t + 3) & 3, (t + 3) & 3, (t + 1) & 3};
}

// TMA descriptors of one sweep direction, one per ring buffer (kernel parameter, __grid_constant__: the kernel
// picks prev / cur / out by the roles of its half-step).
struct SweepMaps {
    CUtensorMap load[4];    // field as the sweep's load box sees it
    CUtensorMap store[4];   // x sweep: one warp's unit [32 rows][U points]
    CUtensorMap edge[4];    // x sweep: 16-byte neighbour boxes
};

constexpr int SLOTS = 64;   // half-steps per chunk of the step loop (work-queue / early-start counters per slot)

struct SweepArgs {
    const double* table;   // device, ROW_DOUBLES per half-step (or per period, see table_period)
    int table_period;      // 0: one row per half-step; p > 0: the rows repeat with period p (constant c and g)
    const int* d_k;        // device: completed solves at the start of the chunk
    int n_off;             // half-step index = n_off + 2 * (*d_k); n_off < SLOTS is also the counter slot
    int ring;              // 3 or 4 field buffers (see roles_of)
    void* bufs[4];         // the ring (y sweep: direct stores into bufs[out])
    int n;                 // unknowns per line
    int nlines;            // number of lines
    int nbk;               // carry series length in units (<= NW, <= NBK_MAX)
    int kb;                // units [0, kb) use the boundary pivots of the table
    const Piece* pieces;   // device
    int npieces;           // all pieces
    int nstatic;           // pieces [0, nstatic) are dealt out statically, the rest through the ticket counter
    const int* cta_off;    // device: CTA b first works pieces [cta_off[b], cta_off[b+1])
    int* tickets;          // device: one zeroed counter per slot of the chunk (indexed by n_off)
    int* done;             // device: one zeroed counter per slot: CTAs whose static share is complete and visible
    int signal;            // 1: the next sweep has safe pieces, so this one publishes `done`
    int early;             // 1: the previous kernel in the stream is sweep nh - 1 of this handle (see "early start")
    int prev_grid;         // its grid size
    long long pitch;       // row pitch in elements
    const void* src;       // compact source window, [p - sp0][line - sl0] (line fastest), or NULL
    int sl0, snl, sp0, snp;
    double g2;             // 2 gamma
    unsigned long long* trace;   // NULL, or [grid][16]: CTA start ns, end ns, SM id, wait cycles, phase cycles of the first and last warp
};

// UT = points per thread ("unit"), NW = consumer warps = units per stage, NSTAGE = TMA stages in flight.
// ONE: the right-hand side is the single input field itself (scheme 1's y sweep, (I - ay+ Dy) U = V): one field per stage.
template <typename T, int DIR, int UT, int NW, int NSTAGE, bool ONE = false>
struct PanelCfg {
    static constexpr int U = UT;                                      // points per unit
    static constexpr int TL = 32;                                     // lines per panel, one per lane
    static constexpr int V = 16 / (int)sizeof(T);                     // elements per 16 bytes
    static constexpr int TU = 128 / (int)sizeof(T);                   // x sweep: points per 128-byte load tile row
    static constexpr int SUB = DIR == 0 ? TU / UT : 1;                // x sweep: units (warps) sharing a load tile
    static constexpr int NT = NW / SUB;                               // x sweep: load tiles per stage and field
    static constexpr int RB = UT * (int)sizeof(T);                    // x sweep: bytes per row of a warp's store tile
    // x sweep: per field NT tiles [32 rows][128 B] (128B-swizzled) + two edge boxes [32 rows][16 B] of wp
    // y sweep: per field one box [U*NW + 2 rows][32 columns]
    static constexpr int HALO = ONE ? 0 : 1;                          // y sweep: stencil rows above / below a stage
    static constexpr int FIELD_BYTES = DIR == 0 ? NT * 4096 : (U * NW + 2 * HALO) * TL * (int)sizeof(T);
    static constexpr int EDGE_BYTES = DIR == 0 ? 512 : 0;
    static constexpr int NFIELDS = ONE ? 1 : 2;
    static constexpr int STAGE_BYTES = NFIELDS * FIELD_BYTES + 2 * EDGE_BYTES;
    static_assert(!ONE || DIR == 1, "single-input variant exists for the y sweep only");
    static constexpr int OUT_BYTES = DIR == 0 ? NW * 2 * 32 * RB : 0;   // two store tiles per warp
    static constexpr int BAR_BYTES = ((NSTAGE * 8) + 15) / 16 * 16;
    static constexpr int TAB_BYTES = 2 * KMAX * (int)sizeof(T);
    static constexpr int XCH_BYTES = (4 * NW * TL + 4 * NW + UT) * (int)sizeof(T);   // L, H [2NW][32]; A, AH [2NW]; pw[UT]
    static constexpr int SMEM_BYTES = 1024 + NSTAGE * STAGE_BYTES + OUT_BYTES + BAR_BYTES + TAB_BYTES + XCH_BYTES;
    static constexpr int THREADS = 32 * NW;
    static_assert((NW & (NW - 1)) == 0, "NW must be a power of two (ring indexing)");
    static_assert(DIR == 1 || (TU % UT == 0 && NW % SUB == 0 && RB >= 32), "x sweep: units must tile the 128-byte row");
    static_assert(FIELD_BYTES % 128 == 0 && (32 * RB) % 1024 == 0 || DIR == 1, "TMA smem alignment");
    static_assert(DIR == 0 || U * NW + 2 * HALO <= 256, "TMA box dimension limit");
};

// ---- x sweep shared-memory tiles ---------------------------------------------------------------------
// Load tile [32 rows][128 B], 128B-swizzled by TMA: 16-byte chunk c of row t sits at chunk c ^ (t & 7).
template <typename T>
__device__ __forceinline__ T tile_elem_x(const unsigned char* tile, int lane, int idx)
{
    const int byte = idx * (int)sizeof(T);
    return *reinterpret_cast<const T*>(tile + lane * 128 + ((((byte >> 4) ^ lane) & 7) << 4) + (byte & 15));
}
// this lane's UT points of sub-unit `sub` of its row
template <typename T, int UT>
__device__ __forceinline__ void load_unit_x(const unsigned char* tile, int lane, int sub, T (&v)[UT])
{
    constexpr int V = 16 / (int)sizeof(T), NC = UT / V;
    const unsigned char* row = tile + lane * 128;
    const int c0 = sub * NC;
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        const unsigned char* p = row + ((((c0 + c) ^ lane) & 7) << 4);
        if constexpr (sizeof(T) == 8) {
            const double2 t = *reinterpret_cast<const double2*>(p);
            v[2 * c] = t.x;
            v[2 * c + 1] = t.y;
        } else {
            const float4 t = *reinterpret_cast<const float4*>(p);
            v[4 * c] = t.x;
            v[4 * c + 1] = t.y;
            v[4 * c + 2] = t.z;
            v[4 * c + 3] = t.w;
        }
    }
}
// Store tile of one warp, [32 rows][RB bytes], swizzled as TMA expects for a box of RB-byte rows
// (128B / 64B / 32B mode: address bits [4,7) ^= bits [7,10), restricted to the row span).
template <typename T, int UT>
__device__ __forceinline__ void store_unit_x(unsigned char* tile, int lane, const T (&v)[UT])
{
    constexpr int V = 16 / (int)sizeof(T), NC = UT / V, RB = UT * (int)sizeof(T);
    unsigned char* row = tile + lane * RB;
    const int f = RB == 128 ? (lane & 7) : RB == 64 ? ((lane >> 1) & 3) : ((lane >> 2) & 1);
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        unsigned char* p = row + ((c ^ f) << 4);
        if constexpr (sizeof(T) == 8)
            *reinterpret_cast<double2*>(p) = make_double2(v[2 * c], v[2 * c + 1]);
        else
            *reinterpret_cast<float4*>(p) = make_float4(v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]);
    }
}

__device__ __forceinline__ void named_bar_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// ---------------------------------------------------------------------------------------------------
// Panel sweep: RHS assembly (A1/A3) fused with the line solve (A2/A4), SURVEY.md 8a.
//   grid  = persistent CTAs (SM count x CTAs/SM); CTA b walks its host-planned pieces.
//   block = NW warps.  Per stage, warp w owns unit g = gbase + s*NW + w (UT points) of the panel's 32
//           lines, lane = line.  Lane 0 of a few warps requests the stage's TMA boxes (ring of NSTAGE stages).
//   stage:  smem -> registers; RHS + local forward; publish L, A; bar (the slot is free: refill it);
//           carry-in, correct y, local backward; publish head; bar;
//           warps whose look-ahead heads are all in this stage finish and store their unit now, the last
//           few keep it one more stage ("deferred").
// ---------------------------------------------------------------------------------------------------
// SRCM: how the source term q s enters.  1 (every shape): a compact window (config 3's 155^2 points) -- the few units it
// covers load their values where they use them.  2: a source on much of the grid -- every unit requests its values
// before it waits for the stage and calls the next stage's into L2.  0: compiled without a source (none is set; ONE
// never adds one).  The host picks the kernel per launch.
template <typename T, int DIR, int UT, int NW, int NSTAGE, int MINB, bool ONE = false, int SRCM = 1>
__global__ void __launch_bounds__(32 * NW, MINB)
wave2d_sweep_panel(const __grid_constant__ SweepMaps maps, const __grid_constant__ SweepArgs a)
{
    constexpr bool SRC = SRCM != 0 && !ONE, DENSE = SRCM == 2 && !ONE;
    using K = PanelCfg<T, DIR, UT, NW, NSTAGE, ONE>;
    constexpr int U = UT, TL = K::TL, V = K::V, SUB = K::SUB, NT = K::NT, RING = 2 * NW;

    extern __shared__ unsigned char smem_raw[];
    const uint32_t raw32 = smem_u32(smem_raw);
    const uint32_t pad = ((raw32 + 1023u) & ~1023u) - raw32;
    unsigned char* sm = smem_raw + pad;   // 1024-byte aligned: the 128B-swizzle atom
    const uint32_t sm32 = raw32 + pad;
    const uint32_t bar32 = sm32 + NSTAGE * K::STAGE_BYTES + K::OUT_BYTES;   // full[NSTAGE]
    T* s_cp = reinterpret_cast<T*>(sm + NSTAGE * K::STAGE_BYTES + K::OUT_BYTES + K::BAR_BYTES);
    T* s_inv = s_cp + KMAX;
    T* s_L = s_inv + KMAX;           // [RING][32]  last local y of a unit
    T* s_H = s_L + RING * TL;        // [RING][32]  first local x of a unit
    T* s_A = s_H + RING * TL;        // [RING]      product of the unit's cp
    T* s_pw = s_A + RING;            // [U]         rho^(e+1)
    T* s_AH = s_pw + U;              // [RING]      the same product, published with H (read by the carry from the right,
                                     //             which outlives the stage: s_A is rewritten one barrier earlier)

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nh = a.n_off + 2 * (*a.d_k);
    const double* row = a.table + static_cast<size_t>(a.table_period ? nh % a.table_period : nh) * ROW_DOUBLES;
    const Roles R = roles_of(nh, a.ring);   // descriptor addresses are formed where they are used (three ints live, not four pointers)
#define tm_prev (&maps.load[R.prev])
#define tm_cur (&maps.load[R.cur])
#define tm_out (&maps.store[R.out])
#define tm_edge (&maps.edge[R.prev])

    for (int i = threadIdx.x; i < KMAX; i += K::THREADS) {
        s_cp[i] = static_cast<T>(row[ROW_CP + i]);
        s_inv[i] = static_cast<T>(row[ROW_INVP + i]);
    }
    if (threadIdx.x == 32 % K::THREADS) {
        T pwr = static_cast<T>(row[ROW_RHO]);
        for (int e = 0; e < U; ++e, pwr *= static_cast<T>(row[ROW_RHO])) s_pw[e] = pwr;
    }
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NSTAGE; ++s) mbar_init(bar32 + 8 * s, 1);
        mbar_fence_init();
        tma_prefetch_desc(tm_prev);
        tma_prefetch_desc(tm_cur);
    }
    __syncthreads();

    // ---- work queue: a CTA first works its own share of the pieces, then draws more from the half-step's
    // ticket counter.  Thread 0 draws for the producer cursor into a ring in shared memory; the other threads
    // read an entry only after a CTA barrier.
    constexpr int QR = 16;
    __shared__ int s_q[QR];
    // Everything above touched only data no earlier kernel writes (the scalar table, the step counter, which
    // changes between graph launches only).  From here on the fields of the previous half-step are read.
    pdl_launch_dependents();
    int* const ticket = a.tickets + a.n_off;
    int own_next = a.cta_off[blockIdx.x];
    const int own_end = a.cta_off[blockIdx.x + 1], nstatic = a.nstatic;
    auto draw = [&]() -> int {   // thread 0: the next piece of this CTA: its own share first, then the queue
        if (own_next < own_end) return own_next++;
        return nstatic < a.npieces ? nstatic + atomicAdd(ticket, 1) : nstatic;   // nothing to draw: no round trip
    };
    if (threadIdx.x == 0) s_q[0] = draw();
    __syncthreads();
    const int npieces = a.npieces;
    // ---- early start.  The previous sweep deals most of its work out statically and finishes the rest in short
    // drawn pieces; its CTAs end several microseconds apart.  A CTA of this kernel that becomes resident meanwhile
    // may already work a "safe" piece: one that reads and writes only lines the previous sweep completed in its
    // static part (the host marks them; a CTA's share is ordered safe-first).  It waits until every CTA of the
    // previous sweep has published "static share complete and visible" (counter `done`), with a time-out after which
    // it simply waits for the whole previous kernel like any unsafe piece does (griddepcontrol.wait).
    bool waited = false;
    {
        const bool try_early = a.early != 0 && s_q[0] < npieces && a.pieces[s_q[0]].safe != 0;
        __shared__ int s_early_ok;
        if (try_early) {
            if (threadIdx.x == 0) {
                const int* flag = a.done + (a.n_off - 1);
                int ok = 0;
                for (int spin = 0; spin < 20000 && !ok; ++spin) {
                    int v;
                    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(flag) : "memory");
                    ok = v >= a.prev_grid;
                    if (!ok) __nanosleep(200);
                }
                s_early_ok = ok;
            }
            __syncthreads();
            if (s_early_ok) asm volatile("fence.proxy.async;" ::: "memory");   // acquired generic writes -> our TMA reads
        }
        if (!try_early || !s_early_ok) {
            pdl_wait();
            waited = true;
        }
    }
    const int nbk = a.nbk, n = a.n, kb = a.kb, nlines = a.nlines;
    const long long pitch = a.pitch;
    [[maybe_unused]] T* const out_lane = reinterpret_cast<T*>(a.bufs[R.out]) + (threadIdx.x & 31);
    unsigned long long t_start = 0;
    if (a.trace && threadIdx.x == 0) t_start = globaltimer_ns();

    // ---- producer cursor (kept by every thread): the next stage to request, NSTAGE ahead of the consumers.
    // The TMA requests of a stage are spread over the warps (lane 0 of each issues its own tile), so that no
    // warp is late at the next barrier; thread 0 posts the stage's byte count on the mbarrier.
    const int sub = DIR == 0 ? warp % SUB : 0, tix = DIR == 0 ? warp / SUB : warp;
    int q_ord = 0, q_s = 0, q_slot = 0;   // ordinal of the producer's piece in this CTA's sequence
    int q_id = s_q[0];
    Piece q_pc = Piece{0, 0, 0, 0};
    if (q_id < npieces) q_pc = a.pieces[q_id];
    // Only the warps that issue a TMA request keep the producer cursor (x: four of them, y: two, ONE: one); the others
    // skip the bookkeeping.  Their own global writes follow a stage's arrival, i.e. the issuing warp's wait on the
    // previous sweep, so they need no griddepcontrol.wait of their own before the end of the kernel.
    const bool producer = DIR == 0 ? warp % (NW / 4) == 0 : ONE ? warp == 0 : warp % (NW / 2) == 0;
    auto produce = [&]() {   // request the next stage into slot q_slot (which must be free)
        if (!producer || q_id >= npieces) return;
        if (lane == 0) {
            const int line0 = q_pc.panel * TL;
            const int g0 = (max(q_pc.ua - nbk, 0) & ~(SUB - 1)) + q_s * NW;
            const uint32_t full = bar32 + 8 * q_slot;
            const uint32_t dst = sm32 + q_slot * K::STAGE_BYTES;
            if (warp == 0) mbar_arrive_expect_tx(full, K::STAGE_BYTES);
            if constexpr (DIR == 0) {
                // fields: one 3D box each, [NT tiles][32 rows][128 B] = 1 KB contiguous per row in global memory
                if (warp == 0) tma_load_3d(dst, tm_prev, 0, line0, g0 / SUB, full);
                if (warp == NW / 2) tma_load_3d(dst + K::FIELD_BYTES, tm_cur, 0, line0, g0 / SUB, full);
                if (warp == NW / 4)
                    tma_load_2d(dst + 2 * K::FIELD_BYTES, tm_edge, g0 * U - V, line0, full);
                if (warp == 3 * NW / 4)
                    tma_load_2d(dst + 2 * K::FIELD_BYTES + K::EDGE_BYTES, tm_edge, (g0 + NW) * U, line0, full);
            } else {
                constexpr int VEC = std::is_same<T, vec2f>::value ? 2 : 1;   // tensor-map columns per lane
                if constexpr (ONE) {
                    if (warp == 0) tma_load_2d(dst, tm_cur, line0 * VEC, g0 * U, full);
                } else {
                    if (warp == 0) tma_load_2d(dst, tm_prev, line0 * VEC, g0 * U - 1, full);
                    if (warp == NW / 2) tma_load_2d(dst + K::FIELD_BYTES, tm_cur, line0 * VEC, g0 * U - 1, full);
                }
            }
        }
        q_slot = q_slot + 1 == NSTAGE ? 0 : q_slot + 1;
        if (++q_s == q_pc.nst) {
            q_s = 0;
            ++q_ord;
            q_id = s_q[q_ord & (QR - 1)];
            if (q_id < npieces) q_pc = a.pieces[q_id];
            if (!waited && !(q_id < npieces && q_pc.safe)) {   // the next piece needs the whole previous sweep
                pdl_wait();
                waited = true;
            }
        }
    };
    // Thread 0 draws the producer's next piece as late as possible: in the stage whose produce() call finishes
    // the current piece, before that stage's CTA barrier (produce() runs right after it).
    auto will_advance = [&]() -> bool { return q_id < npieces && q_s + 1 == q_pc.nst; };
    auto draw_ahead = [&]() {
        if (threadIdx.x == 0 && will_advance()) s_q[(q_ord + 1) & (QR - 1)] = draw();
    };
#pragma unroll
    for (int s = 0; s < NSTAGE; ++s) {
        draw_ahead();
        __syncthreads();   // (thread 0 may have drawn the next piece)
        produce();
    }

    // ---- consumers (all warps)
    const T rho = static_cast<T>(row[ROW_RHO]), inv = static_cast<T>(row[ROW_INV]);
    const T am = static_cast<T>(row[ROW_AM]), q = static_cast<T>(row[ROW_Q]);
    const T c1 = static_cast<T>(row[ROW_C1]), g2 = static_cast<T>(a.g2);
    const T ami = am * inv, c1i = c1 * inv, g2i = g2 * inv, qi = q * inv;   // stationary rows: r_e inv in one go
    auto cp_at = [&](int p) -> T { return p < KMAX ? s_cp[p] : rho; };
    auto inv_at = [&](int p) -> T { return p < KMAX ? s_inv[p] : inv; };
    auto pw_at = [&](int e) -> T { return s_pw[e]; };   // rho^(e+1), broadcast read

    // warps [0, wdef) finish their unit in the stage that computed it; warps [wdef, NW) one stage later
    const int wdef = ((NW - nbk) / SUB) * SUB;
    [[maybe_unused]] unsigned char* const my_out0 = sm + NSTAGE * K::STAGE_BYTES + warp * (2 * 32 * K::RB);
    [[maybe_unused]] unsigned char* my_out = my_out0;   // alternates between the warp's two store tiles
    const T* const sL_lane = s_L + lane;
    const T* const sH_lane = s_H + lane;

    // carry series: value entering unit `ring` from the left (dirn = -1, over L) or from the right (+1, over H)
    // `stat`: all nbk units of the series are whole units with stationary pivots, so every A is rho^U.
    const T pwU = pw_at(U - 1);
    auto carry = [&](const T* vals_lane, const T* fac, int ring, int dirn, bool stat) -> T {
        T c = T(0);
        if (stat) {
            if (nbk > 4) {
#pragma unroll
                for (int j = NBK_MAX; j > 4; --j)
                    if (j <= nbk) c = fmaT(pwU, c, vals_lane[((ring + dirn * j) & (RING - 1)) * TL]);
            }
#pragma unroll
            for (int j = 4; j >= 1; --j)
                if (j <= nbk) c = fmaT(pwU, c, vals_lane[((ring + dirn * j) & (RING - 1)) * TL]);
            return c;
        }
        if (nbk > 4) {
#pragma unroll
            for (int j = NBK_MAX; j > 4; --j)
                if (j <= nbk) {
                    const int idx = (ring + dirn * j) & (RING - 1);
                    c = fmaT(fac[idx], c, vals_lane[idx * TL]);
                }
        }
#pragma unroll
        for (int j = 4; j >= 1; --j)
            if (j <= nbk) {
                const int idx = (ring + dirn * j) & (RING - 1);
                c = fmaT(fac[idx], c, vals_lane[idx * TL]);
            }
        return c;
    };

    // finish unit gp (local x in v[]): add the carry from the right, store
    auto finish = [&](T (&v)[U], int gp, int ring, const Piece& pc) {
        const T Xin = carry(sH_lane, s_AH, ring, +1, gp + 1 >= kb && (gp + nbk + 1) * U <= n);   // x at the start of unit gp+1
        if (gp < pc.ua || gp >= pc.ub) return;    // warp-uniform
        const int pp0 = gp * U;
        const bool full = pp0 + U <= n;
        if (gp >= kb && full) {
#pragma unroll
            for (int e = 0; e < U; ++e) v[e] = fmaT(pw_at(U - 1 - e), Xin, v[e]);
        } else {
            T c = Xin;
#pragma unroll
            for (int e = U - 1; e >= 0; --e) {
                c *= cp_at(pp0 + e);
                v[e] += c;
            }
        }
        if constexpr (DIR == 0) {
            if (lane == 0) tma_wait_read<1>();   // the store before the previous one has read this tile
            __syncwarp();
            store_unit_x<T, U>(my_out, lane, v);
            fence_async_smem();
            __syncwarp();
            if (lane == 0) {
                tma_store_2d(tm_out, pp0, pc.panel * TL, smem_u32(my_out));
                tma_commit();
            }
            my_out = my_out == my_out0 ? my_out0 + 32 * K::RB : my_out0;
        } else {
            if (pc.panel * TL + lane < nlines) {
                T* o = out_lane + pc.panel * TL + static_cast<long long>(pp0) * pitch;
                if (full) {
#pragma unroll
                    for (int e = 0; e < U; ++e, o += pitch) *o = v[e];
                } else {
#pragma unroll
                    for (int e = 0; e < U; ++e, o += pitch)
                        if (pp0 + e < n) *o = v[e];
                }
            }
        }
    };

    int slot = 0, phase = 0;

    // The stage loop, compiled twice: DEF = false for warps that finish their unit in the same stage,
    // DEF = true for the last few warps, which keep the local x of their unit in registers for one stage.
    // "static share complete": every warp makes its own stores visible (x sweep: its TMA stores have completed;
    // y sweep: fence), then after the next CTA barrier thread 0 counts the CTA in `done` (release).
    const int own_count = own_end - a.cta_off[blockIdx.x];
    bool signaled = a.signal == 0, signaled_now = false;   // nothing to publish if nobody will look
    auto publish_static_done = [&]() {
        if constexpr (DIR == 0) {
            if (lane == 0) tma_wait_all();
        }
        __threadfence();
        signaled_now = true;
    };
    auto run_pieces = [&](auto def_c) {
        constexpr bool DEF = decltype(def_c)::value;
        T pend[DEF ? U : 1];
#pragma unroll
        for (int e = 0; e < (DEF ? U : 1); ++e) pend[e] = T(0);

        for (int ord = 0;; ++ord) {
            const int pid = s_q[ord & (QR - 1)];
            if (pid >= npieces) break;
            const Piece pc = a.pieces[pid];
            const int line0 = pc.panel * TL, line = line0 + lane;
            const int gbase = max(pc.ua - nbk, 0) & ~(SUB - 1);
            [[maybe_unused]] const bool src_tile = SRC && a.src != nullptr && line0 < a.sl0 + a.snl && line0 + TL > a.sl0;
            [[maybe_unused]] const bool src_line = SRC && line >= a.sl0 && line < a.sl0 + a.snl;
            [[maybe_unused]] const T* srcp = reinterpret_cast<const T*>(a.src) + (line - a.sl0);

            if (!signaled && ord > own_count) {   // static share and one drawn piece done: its stores have landed
                publish_static_done();
                signaled = true;
            }
            named_bar_sync(1, NW * 32);   // the previous piece is completely finished
            if (signaled_now) {
                if (threadIdx.x == 0) {
                    __threadfence();
                    atomicAdd(a.done + a.n_off, 1);
                }
                signaled_now = false;
            }
            s_L[(NW + warp) * TL + lane] = T(0);   // "stage -1": zero carries
            if (lane == 0) s_A[NW + warp] = T(0);

            // The stages of the piece.  (Two copies, with and without the source term, chosen per piece by whether its lines
            // meet a compact window, were measured: 140.5 instead of 130.3 us per step at config 3 -- the instruction
            // cache pays more than the leaner loop saves.)
            auto stages = [&](auto src_c) {
                constexpr bool PSRC = decltype(src_c)::value, PDENSE = PSRC && DENSE;
                for (int s = 0; s < pc.nst; ++s) {
                    const int ring = (s & 1) * NW + warp;
                    const int g = gbase + s * NW + warp, p0 = g * U;
                    T xl[U];
                    // ---- source values of this unit (a source window that covers it: rare with a compact window, every unit
                    // with a dense s): requested before the stage's data is awaited, used at the end of the right-hand side
                    [[maybe_unused]] bool src_unit = false;
                    [[maybe_unused]] T sv[PDENSE ? U : 1];
                    if constexpr (PSRC) src_unit = src_tile && src_line && p0 < a.sp0 + a.snp && p0 + U > a.sp0;
                    if constexpr (PDENSE) {
                        if (src_unit) {
    #pragma unroll
                            for (int e = 0; e < U; ++e) {
                                const int ps = p0 + e - a.sp0;
                                sv[e] = ps >= 0 && ps < a.snp && p0 + e < n ? srcp[static_cast<size_t>(ps) * a.snl] : T(0);
                            }
                        }
                        if (src_tile && src_line && (lane & 15) == 0) {   // and the next stage's lines of s are called into L2
                            const int ps0 = p0 + NW * U - a.sp0;
    #pragma unroll
                            for (int e = 0; e < U; ++e)
                                if (ps0 + e >= 0 && ps0 + e < a.snp) prefetch_l2(srcp + static_cast<size_t>(ps0 + e) * a.snl);
                        }
                    }
                    // ---- shared memory -> registers
                    mbar_wait(bar32 + 8 * slot, phase);
                    draw_ahead();   // (thread 0) the ticket's round trip overlaps this stage's first half
                    const unsigned char* st = sm + slot * K::STAGE_BYTES;
                    if (++slot == NSTAGE) { slot = 0; phase ^= 1; }
                    [[maybe_unused]] T wp[U], wl, wr;
                    T wc[U];
                    if constexpr (DIR == 0) {
                        const unsigned char* tp = st + tix * 4096;
                        load_unit_x<T, U>(tp, lane, sub, wp);
                        load_unit_x<T, U>(tp + K::FIELD_BYTES, lane, sub, wc);
                        if (sub > 0) wl = tile_elem_x<T>(tp, lane, sub * U - 1);
                        else if (tix > 0) wl = tile_elem_x<T>(tp - 4096, lane, K::TU - 1);
                        else wl = reinterpret_cast<const T*>(st + 2 * K::FIELD_BYTES)[lane * V + V - 1];
                        if (sub < SUB - 1) wr = tile_elem_x<T>(tp, lane, (sub + 1) * U);
                        else if (tix < NT - 1) wr = tile_elem_x<T>(tp + 4096, lane, 0);
                        else wr = reinterpret_cast<const T*>(st + 2 * K::FIELD_BYTES + K::EDGE_BYTES)[lane * V];
                    } else if constexpr (ONE) {
                        const T* ccv = reinterpret_cast<const T*>(st) + (warp * U) * TL + lane;
    #pragma unroll
                        for (int e = 0; e < U; ++e) wc[e] = ccv[e * TL];
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
                    // ---- RHS + local forward elimination
                    const bool fast = g >= kb && p0 + U <= n;   // stationary pivots, whole unit inside the line
                    T Aval;
                    if (fast) {   // y_e = rho y_{e-1} + inv r_e from y_{-1} = 0
    #pragma unroll
                        for (int e = 0; e < U; ++e) {
                            if constexpr (ONE) {
                                xl[e] = inv * wc[e];
                            } else {
                                const T left = e == 0 ? wl : wp[e - 1];
                                const T right = e == U - 1 ? wr : wp[e + 1];
                                xl[e] = fmaT(g2i, wc[e], fmaT(ami, left + right, c1i * wp[e]));
                            }
                        }
                        if constexpr (PDENSE) {
                            if (src_unit) {
    #pragma unroll
                                for (int e = 0; e < U; ++e) xl[e] = fmaT(qi, sv[e], xl[e]);
                            }
                        } else if constexpr (PSRC) {
                            if (src_unit) {
    #pragma unroll
                                for (int e = 0; e < U; ++e) {
                                    const int ps = p0 + e - a.sp0;
                                    if (ps >= 0 && ps < a.snp) xl[e] = fmaT(qi, srcp[static_cast<size_t>(ps) * a.snl], xl[e]);
                                }
                            }
                        }
    #pragma unroll
                        for (int e = 1; e < U; ++e) xl[e] = fmaT(rho, xl[e - 1], xl[e]);
                        Aval = pw_at(U - 1);
                    } else {
                        T fy = T(0), prod = T(1);
    #pragma unroll
                        for (int e = 0; e < U; ++e) {
                            const int p = p0 + e;
                            T r;
                            if constexpr (ONE) {
                                r = wc[e];
                            } else {
                                const T left = e == 0 ? wl : wp[e - 1];
                                const T right = e == U - 1 ? wr : wp[e + 1];
                                r = fmaT(g2, wc[e], fmaT(am, left + right, c1 * wp[e]));
                            }
                            if constexpr (PDENSE) {
                                if (src_unit) r = fmaT(q, sv[e], r);
                            } else if constexpr (PSRC) {
                                if (src_unit && p >= a.sp0 && p < a.sp0 + a.snp)
                                    r = fmaT(q, srcp[static_cast<size_t>(p - a.sp0) * a.snl], r);
                            }
                            const T cpe = cp_at(p);
                            fy = fmaT(cpe, fy, r * inv_at(p));
                            if (p >= n) fy = T(0);
                            prod *= cpe;
                            xl[e] = fy;
                        }
                        Aval = prod;
                    }
                    s_L[ring * TL + lane] = xl[U - 1];
                    if (lane == 0) s_A[ring] = Aval;
                    named_bar_sync(1, NW * 32);
                    produce();   // every warp holds its stage data in registers: refill the slot

                    // ---- carry from the left, local back substitution
                    const T Yin = carry(sL_lane, s_A, ring, -1, g - nbk >= kb && p0 <= n);   // y at the end of unit g-1
                    if (fast) {
                        xl[U - 1] = fmaT(pw_at(U - 1), Yin, xl[U - 1]);
    #pragma unroll
                        for (int e = U - 2; e >= 0; --e) xl[e] = fmaT(rho, xl[e + 1], fmaT(pw_at(e), Yin, xl[e]));
                    } else {
                        T c = Yin;
    #pragma unroll
                        for (int e = 0; e < U; ++e) {
                            c *= cp_at(p0 + e);
                            xl[e] = p0 + e < n ? xl[e] + c : T(0);
                        }
    #pragma unroll
                        for (int e = U - 2; e >= 0; --e) xl[e] = fmaT(cp_at(p0 + e), xl[e + 1], xl[e]);
                    }
                    s_H[ring * TL + lane] = xl[0];
                    if (lane == 0) s_AH[ring] = Aval;
                    named_bar_sync(1, NW * 32);

                    // ---- carry from the right, store
                    if constexpr (DEF) {
                        if (s > 0) finish(pend, g - NW, ring ^ NW, pc);
    #pragma unroll
                        for (int e = 0; e < U; ++e) pend[e] = xl[e];
                    } else {
                        finish(xl, g, ring, pc);
                    }
                }
            };
            stages(std::integral_constant<bool, SRC>{});
            // ---- flush: the deferred units of the last stage see zero heads beyond it
            const int ringf = (pc.nst & 1) * NW + warp;
            named_bar_sync(1, NW * 32);   // the deferred warps have read the heads of stage nst-2 (same half of the ring)
            s_H[ringf * TL + lane] = T(0);
            if (lane == 0) s_AH[ringf] = T(0);   // (a one-stage piece never wrote this half: keep 0 * AH finite)
            named_bar_sync(1, NW * 32);
            if constexpr (DEF) {
                if (pc.nst > 0) finish(pend, gbase + (pc.nst - 1) * NW + warp, ringf ^ NW, pc);
            }
        }
    };
    if (warp >= wdef) run_pieces(std::true_type{});
    else run_pieces(std::false_type{});

    if (!waited) pdl_wait();   // (a CTA whose pieces were all safe) never exit before the previous kernel has
    if (!signaled) {           // few or no drawn pieces: publish at the end
        publish_static_done();
        named_bar_sync(1, NW * 32);
        if (threadIdx.x == 0) {
            __threadfence();
            atomicAdd(a.done + a.n_off, 1);
        }
    }
    if constexpr (DIR == 0) {
        if (lane == 0) tma_wait_read<0>();
    }
    if (a.trace) {
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned long long* t = a.trace + 16 * static_cast<size_t>(blockIdx.x);
            t[0] = t_start;
            t[1] = globaltimer_ns();
            t[2] = smid();
            t[3] = static_cast<unsigned long long>(q_ord);
        }
    }
#undef tm_prev
#undef tm_cur
#undef tm_out
#undef tm_edge
}

struct FieldSet {   // the ring of field buffers; roles by roles_of(nh, ring)
    void* b[4];
    int ring;
};

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

// out = (I - ay Dy) in: in - ay (in[j-1] - 2 in[j] + in[j+1]) with zero ghosts (scheme 1 start, one-time)
template <typename T>
__global__ void wave2d_apply_y(T* __restrict__ out, const T* __restrict__ in, int n1, int n2, long long pitch, double ay)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= n1 || j >= n2) return;
    const long long o = j * pitch + i;
    const T up = j > 0 ? in[o - pitch] : T(0), dn = j < n2 - 1 ? in[o + pitch] : T(0), c0 = in[o];
    out[o] = c0 - static_cast<T>(ay) * (up - T(2) * c0 + dn);
}

// Second-order start of the three-level scheme (2.8) (option "start" = 2, scheme 1; one-time):
// u1 += ax (phi[i-1] - 2 phi + phi[i+1]) + ay (phi[j-1] - 2 phi + phi[j+1]) + qs s,  ax = tau^2 c^0 / (2 h1^2), ay likewise,
// qs = tau^2 g^0 / 2, zero ghosts (2.10); s: compact source window [j - j0][i - i0] or NULL.
template <typename T>
__global__ void wave2d_start2(T* __restrict__ u1, const T* __restrict__ phi, int n1, int n2, long long pitch, double ax,
                              double ay, double qs, const T* __restrict__ s, int i0, int j0, int sw, int sh)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= n1 || j >= n2) return;
    const long long o = j * pitch + i;
    const T c0 = phi[o];
    const T we = i > 0 ? phi[o - 1] : T(0), ea = i < n1 - 1 ? phi[o + 1] : T(0);
    const T so = j > 0 ? phi[o - pitch] : T(0), no = j < n2 - 1 ? phi[o + pitch] : T(0);
    T v = static_cast<T>(ax) * (we - T(2) * c0 + ea) + static_cast<T>(ay) * (so - T(2) * c0 + no);
    if (s != nullptr && i >= i0 && i < i0 + sw && j >= j0 && j < j0 + sh)
        v += static_cast<T>(qs) * s[static_cast<size_t>(j - j0) * sw + (i - i0)];
    u1[o] += v;
}

// dst[p][l] = src[l][p] for a small window (compact source, transposed copy for the x sweep)
template <typename T>
__global__ void wave2d_transpose_small(T* __restrict__ dst, const T* __restrict__ src, int rows, int cols)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x, r = blockIdx.y;
    if (c < cols && r < rows) dst[static_cast<size_t>(c) * rows + r] = src[static_cast<size_t>(r) * cols + c];
}

// End of a chunk of the step loop: count its solves and zero the work-queue / early-start counters it used.
// Launched without programmatic serialization: every sweep of the chunk has completed.
__global__ void wave2d_end_chunk(int* d_k, int by, int* counters)
{
    counters[threadIdx.x] = 0;   // blockDim.x == 2 * SLOTS: tickets | done
    if (threadIdx.x == 0) *d_k += by;
}

}  // namespace w2d
