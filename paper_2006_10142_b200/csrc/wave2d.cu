// wave2d.cu -- C ABI of libwave2d.so (include/wave2d.h): host-side planning, the per-half-step scalar
// table (A0), TMA descriptors, the CUDA-Graph step loop (A6/A7) and the launches of kernels.cuh.
#include "../../include/wave2d.h"

#include <cuda.h>
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>   // header-only: ranges show up in a timeline profiler, cost nothing without one

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "kernels.cuh"
#include "exact.cuh"
#include "line.cuh"

using namespace w2d;

namespace {

// NVTX range for the duration of a scope ("x_sweep" / "y_sweep" around the sweep launches, the API calls by name)
struct Range {
    explicit Range(const char* name) { nvtxRangePushA(name); }
    ~Range() { nvtxRangePop(); }
};

// ------------------------------------------------------------------------------------------------
// Kernel variants: (NW consumer warps = units per stage, NSTAGE) per dtype and direction.
// ------------------------------------------------------------------------------------------------
struct Variant {
    int dir, nw, nstage, unit, sub, smem, threads, elem;   // elem = bytes per grid value, unit = points per thread
    int vec;                                               // grid lines per lane (2: fp32 y sweep on vec2f)
    int one;                                               // 1: single-input y sweep of scheme 1
    const void* fn;
    const void* fn_nosrc;                                  // the same shape compiled without the source term, or NULL
    const void* fn_dense;                                  // ... for a source on much of the grid, or NULL
};

// NOSRC: also instantiate the shape without the source term and for a dense source (the default shapes)
template <typename T, int DIR, int UT, int NW, int NSTAGE, int MINB = 1, bool ONE = false, bool NOSRC = false>
Variant make_variant()
{
    using K = PanelCfg<T, DIR, UT, NW, NSTAGE, ONE>;
    constexpr int VEC = std::is_same<T, vec2f>::value ? 2 : 1;
    const void *nosrc = nullptr, *dense = nullptr;
    if constexpr (NOSRC) {
        nosrc = reinterpret_cast<const void*>(&wave2d_sweep_panel<T, DIR, UT, NW, NSTAGE, MINB, ONE, 0>);
        dense = reinterpret_cast<const void*>(&wave2d_sweep_panel<T, DIR, UT, NW, NSTAGE, MINB, ONE, 2>);
    }
    return Variant{DIR, NW, NSTAGE, UT, K::SUB, K::SMEM_BYTES, K::THREADS, (int)sizeof(T) / VEC, VEC, ONE ? 1 : 0,
                   reinterpret_cast<const void*>(&wave2d_sweep_panel<T, DIR, UT, NW, NSTAGE, MINB, ONE, 1>), nosrc, dense};
}

constexpr int NVAR = 4;   // shape variants per (dtype, dir); index 0 is the default
void add_shapes_f64(std::vector<Variant>& v)
{
    v.push_back(make_variant<double, 0, 8, 16, 2, 1, false, true>());
    v.push_back(make_variant<double, 0, 8, 8, 2, 2>());
    v.push_back(make_variant<double, 0, 16, 8, 2>());
    v.push_back(make_variant<double, 0, 4, 16, 2>());
    v.push_back(make_variant<double, 1, 8, 16, 2, 1, false, true>());
    v.push_back(make_variant<double, 1, 8, 8, 3, 2>());
    v.push_back(make_variant<double, 1, 16, 8, 3>());
    v.push_back(make_variant<double, 1, 8, 16, 3>());
}
void add_shapes_one(std::vector<Variant>& v)   // scheme 1 y sweep; shape index 0..1
{
    v.push_back(make_variant<double, 1, 8, 16, 3, 1, true>());
    v.push_back(make_variant<double, 1, 16, 16, 3, 1, true>());
    v.push_back(make_variant<vec2f, 1, 8, 16, 3, 1, true>());
    v.push_back(make_variant<float, 1, 8, 8, 4, 2, true>());
}
void add_shapes_f32(std::vector<Variant>& v)
{
    v.push_back(make_variant<float, 0, 16, 16, 2, 1, false, true>());
    v.push_back(make_variant<float, 0, 16, 8, 2, 2>());
    v.push_back(make_variant<float, 0, 32, 8, 2>());
    v.push_back(make_variant<float, 0, 8, 16, 2>());
    v.push_back(make_variant<vec2f, 1, 8, 16, 2, 1, false, true>());    // two columns per lane; not with a source (falls to shape 1)
    v.push_back(make_variant<float, 1, 8, 8, 3, 2, false, true>());   // (the fp32 y sweep of a run with a source)
    v.push_back(make_variant<float, 1, 16, 8, 3>());
    v.push_back(make_variant<float, 1, 8, 16, 4>());
}

const std::vector<Variant>& variants()
{
    static std::vector<Variant> v = [] {
        std::vector<Variant> w;
        add_shapes_f64(w);
        add_shapes_f32(w);
        add_shapes_one(w);
        return w;
    }();
    return v;
}

const Variant* find_variant(int elem, int dir, int shape, int one = 0)
{
    int seen = 0;
    for (const Variant& v : variants())
        if (v.elem == elem && v.dir == dir && v.one == one) {
            if (seen == shape) return &v;
            ++seen;
        }
    return nullptr;
}

// ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled()
{
    static EncodeTiledFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) != cudaSuccess) p = nullptr;
        return reinterpret_cast<EncodeTiledFn>(p);
    }();
    return fn;
}

constexpr int MAX_CHUNK = SLOTS / 2;   // time steps in the longest chunk of the step loop (32)
constexpr int NCHUNK = 6;              // chunk lengths 1, 2, 4, 8, 16, 32
static_assert((1 << (NCHUNK - 1)) == MAX_CHUNK, "chunk lengths are the powers of two up to MAX_CHUNK");

struct DirPlan {
    int solver = WAVE2D_SOLVER_STREAM;   // STREAM or EXACT after planning
    int nbk = 1, kb = 0, halo = 0, shape = 0;
    double rho = 0.0;
    const Variant* var = nullptr;
    int n = 0, nlines = 0, npanels = 0, total_units = 0, grid = 0, ctas_per_sm = 0, quota = 0;
    std::vector<Piece> pieces;
    std::vector<int> cta_off;   // CTA b's static share: pieces [cta_off[b], cta_off[b+1]); pieces >= nstatic are drawn
    int nstatic = 0;
    bool has_safe = false;      // some static piece may start before the previous sweep ends (early start)
    // exact path (exact.cuh)
    const void* ex_fn = nullptr;
    int ex_wpc = 0, ex_nseg = 0, ex_sc = 0, ex_smem = 0;
};

}  // namespace

struct wave2d_s {
    int N1, N2, n1, n2, M, dtype, elem;
    double l, tau, gamma = 2.0, kappa = 0.5, sigma = 0.5;
    double ly = 0.0;                     // > 0: extent in y of THIS grid (h2 = ly / N2): a row block of a larger domain
    int opt_start = 1;                   // scheme 1: 1 = (2.9) as printed, 2 = second-order start
    int opt_solver = WAVE2D_SOLVER_AUTO, opt_graph = 1, opt_graph_steps = MAX_CHUNK, opt_shape[2] = {0, 0};
    int opt_quota[2] = {0, 0};
    cudaStream_t own_stream = nullptr, stream = nullptr;
    int num_sms = 0;

    long long pitch = 0;                 // elements
    int scheme = 0;                      // 0: split scheme (2.11)-(2.12); 1: factorised unsplit scheme (2.8)
    bool v_ready = false;                // scheme 1: V^0, V^1 computed from U^0, U^1 (needs the final c samples)
    void* buf[4] = {nullptr, nullptr, nullptr, nullptr};   // scheme 0 uses 3
    bool ext_fields = false;             // the ring lives in caller memory (wave2d_set_workspace): never freed here
    std::vector<double> c_half, g_half;  // g_half empty: g == 1
    bool have_cs = false;                // spatial speed factor set (wave2d_set_speed_field): variable-coefficient solvers
    void* d_cs = nullptr;                // pitched like a field, pad 0
    bool have_src = false;
    void* src_dev[2] = {nullptr, nullptr};    // [0]: x sweep (transposed window), [1]: y sweep (natural window)
    int win_i0 = 0, win_j0 = 0, win_w = 0, win_h = 0;

    std::vector<double> table;           // host copy
    int table_period = 0;                // 0: one row per half-step; 2: constant c and g, two rows serve every step
    double* d_table = nullptr;
    size_t table_bytes = 0, pieces_bytes[2] = {0, 0}, cta_off_bytes[2] = {0, 0}, trace_bytes[2] = {0, 0};
    int* d_k = nullptr;
    bool plan_ok = false;
    DirPlan plan[2];
    bool line_mode = false;              // small grid: the step loop runs in wave2d_line_steps (line.cuh)
    bool line_resident = false;          // ... in wave2d_line_resident: the fields stay in the cluster's shared memory
    int opt_resident = 1;
    const void* line_fn = nullptr;
    int line_unit = 0, line_ctas = 0, line_smem = 0;
    SweepMaps maps[2];                   // per direction: TMA descriptors of every ring buffer
    Piece* d_pieces[2] = {nullptr, nullptr};
    int* d_tickets = nullptr;              // tickets[SLOTS] | done[SLOTS]: per slot of a chunk, zeroed by wave2d_end_chunk
    int* d_cta_off[2] = {nullptr, nullptr};
    double opt_static_frac = -1.0, opt_tail_div = 2.0;   // static_frac < 0: by dtype (plan_dir)
    int opt_tail_min = 0, opt_tail_max = 6;   // tail_min 0: planned from the stage size
    int opt_trace = 0, opt_pdl = 1, opt_early = 1;
    unsigned long long* d_trace[2] = {nullptr, nullptr};   // per-CTA trace of the last launch per direction
    cudaGraphExec_t gexec[NCHUNK] = {};   // gexec[i]: a chunk of 2^i time steps (built with the plan)

    bool have_initial = false, ran = false;
    int k = 0;                           // completed steps
    long long launches = 0;              // kernels launched (graph nodes count individually)
    long long graph_launches = 0;        // cudaGraphLaunch calls
    long long plain_sweeps = 0;          // sweep kernels launched outside a graph
    long long line_launches = 0;         // launches of the small-grid step kernel
    size_t device_bytes = 0;
    std::string err;
};

namespace {

double step_y(const wave2d_t* h) { return (h->ly > 0.0 ? h->ly : h->l) / h->N2; }

#define W2D_CUDA(h, call)                                                                      \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) {                                                               \
            (h)->err = std::string(#call) + ": " + cudaGetErrorString(e_);                     \
            (void)cudaGetLastError();                                                          \
            return WAVE2D_ERR_CUDA;                                                            \
        }                                                                                      \
    } while (0)

int dev_alloc(wave2d_t* h, void** p, size_t bytes)
{
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) {
        h->err = std::string("cudaMalloc: ") + cudaGetErrorString(e);
        (void)cudaGetLastError();
        *p = nullptr;
        return WAVE2D_ERR_ALLOC;
    }
    h->device_bytes += bytes;
    return WAVE2D_OK;
}

void dev_free(wave2d_t* h, void* p, size_t bytes)
{
    if (!p) return;
    cudaFree(p);
    h->device_bytes -= bytes;
}

void drop_graph(wave2d_t* h)
{
    for (cudaGraphExec_t& g : h->gexec) {
        if (g) cudaGraphExecDestroy(g);
        g = nullptr;
    }
}

void invalidate_plan(wave2d_t* h)
{
    h->plan_ok = false;
    drop_graph(h);
}

// ---- A0: per-half-step scalars, fp64 on the host -----------------------------------------
// One table row: half-step with alpha+ = ap, alpha- = am, source factor qv (0 without a source).
void fill_row(double* row, double gamma, double ap, double am, double qv)
{
    const double beta = gamma + 2.0 * ap;
    const double rho = 2.0 * ap / (beta + std::sqrt(beta * beta - 4.0 * ap * ap));   // small root of ap z^2 - beta z + ap
    row[ROW_AM] = am;
    row[ROW_Q] = qv;
    row[ROW_RHO] = rho;
    row[ROW_INV] = 1.0 / (beta - ap * rho);
    row[ROW_C1] = -(gamma + 2.0 * am);
    row[ROW_AP] = ap;
    row[ROW_BETA] = beta;
    row[ROW_LNR] = std::log(rho);
    double cp = 0.0;
    for (int p = 0; p < KMAX; ++p) {   // LU pivots of tridiag(-ap, beta, -ap): inv_p = 1/u_pp, cp_p = ap/u_pp
        const double iv = 1.0 / (beta - ap * cp);
        cp = ap * iv;
        row[ROW_CP + p] = cp;
        row[ROW_INVP + p] = iv;
    }
}

void build_table(wave2d_t* h)
{
    // Constant c and g (the paper's own runs): all x rows are equal and all y rows are equal, so two rows
    // serve every step and M is not bounded by the size of the table.
    bool constant = h->M >= 2;
    for (size_t i = 1; i < h->c_half.size() && constant; ++i) constant = h->c_half[i] == h->c_half[0];
    if (h->have_src)
        for (size_t i = 1; i < h->g_half.size() && constant; ++i) constant = h->g_half[i] == h->g_half[0];
    h->table_period = constant ? 2 : 0;
    const int nhalf = constant ? 2 : 2 * h->M;
    h->table.assign(static_cast<size_t>(std::max(nhalf, 1)) * ROW_DOUBLES, 0.0);
    const double t2 = h->tau * h->tau;
    if (h->scheme == 1) {
        // Factorised (2.8): step k -> k+1 (k = t + 1) is sweep 2t (x) and 2t+1 (y), both with
        // gamma = 1:  x: (I - ax+ Dx) V^{k+1} = 2 U^k - (I - ax- Dx) V^{k-1} + tau^2 g_k s,  y: (I - ay+ Dy) U^{k+1} = V^{k+1}
        // (V^j = (I - ay(c^j) Dy) U^j is carried); a_d^+- = tau^2 c^{k+-1} / (2 h_d^2).
        for (int t = 0; t + 2 <= (constant ? 2 : h->M); ++t) {
            const int k = t + 1;
            const double h1 = h->l / h->N1, h2 = step_y(h);
            const double cp1 = h->c_half[2 * (k + 1)], cm1 = h->c_half[2 * (k - 1)];
            const double g = h->g_half.empty() ? 1.0 : h->g_half[2 * k];
            fill_row(&h->table[static_cast<size_t>(2 * t) * ROW_DOUBLES], 1.0, t2 * cp1 / (2.0 * h1 * h1),
                     t2 * cm1 / (2.0 * h1 * h1), h->have_src ? t2 * g : 0.0);
            fill_row(&h->table[static_cast<size_t>(2 * t + 1) * ROW_DOUBLES], 1.0, t2 * cp1 / (2.0 * h2 * h2), 0.0, 0.0);
        }
        return;
    }
    for (int n = 0; n < nhalf; ++n) {
        const double hd = (n & 1) == 0 ? h->l / h->N1 : step_y(h);                    // reading R3
        // sigma = 1/2: (2.11)-(2.12); sigma = 1: the fully implicit weights of Listing 1
        const double ap = h->sigma * t2 * h->c_half[n + 1] / (hd * hd);
        const double am = (1.0 - h->sigma) * t2 * h->c_half[n > 0 ? n - 1 : 0] / (hd * hd);   // reading R5: c_{-1} := c_0
        const double g = h->g_half.empty() ? 1.0 : h->g_half[n];                   // reading R8
        fill_row(&h->table[static_cast<size_t>(n) * ROW_DOUBLES], h->gamma, ap, am, h->have_src ? h->kappa * t2 * g : 0.0);
    }
}

// swizzle: 0 (none) or the row span in bytes of the swizzle mode (32 / 64 / 128)
int make_tmap(wave2d_t* h, CUtensorMap* tm, void* base, int box0, int box1, int swizzle)
{
    EncodeTiledFn enc = encode_tiled();
    if (!enc) {
        h->err = "cuTensorMapEncodeTiled entry point not available";
        return WAVE2D_ERR_CUDA;
    }
    const cuuint64_t dims[2] = {(cuuint64_t)h->n1, (cuuint64_t)h->n2};
    const cuuint64_t strides[1] = {(cuuint64_t)h->pitch * h->elem};
    const cuuint32_t box[2] = {(cuuint32_t)box0, (cuuint32_t)box1};
    const cuuint32_t es[2] = {1, 1};
    CUresult r = enc(tm, h->dtype == WAVE2D_F64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2,
                     base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     swizzle == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : swizzle == 64 ? CU_TENSOR_MAP_SWIZZLE_64B
                     : swizzle == 32 ? CU_TENSOR_MAP_SWIZZLE_32B : CU_TENSOR_MAP_SWIZZLE_NONE,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        char msg[160];
        snprintf(msg, sizeof msg, "cuTensorMapEncodeTiled failed (%d) box=%dx%d n=%dx%d pitch=%lld", (int)r, box0, box1,
                 h->n1, h->n2, h->pitch);
        h->err = msg;
        return WAVE2D_ERR_CUDA;
    }
    return WAVE2D_OK;
}

// Cut the (panel, unit) space into pieces of work (panel-major).  A cut costs 2 nbk extra units (carry warm-up
// before the cut, look-ahead after it).  The first part of the space is dealt out statically, `quota` stages to
// each of `slots` CTAs (cta_off); the rest is cut into short pieces that the CTAs draw from an atomic ticket
// counter once their own share is done, so that CTAs the memory system serves more slowly get less of it.  The
// short pieces follow guided self-scheduling (remaining / (2 slots) stages, between 2 and 6).
// `fixed` > 0 (tests): no static part, every piece `fixed` stages long.
void build_pieces(DirPlan& P, int nw, int sub, int slots, int fixed, double static_frac, int tail_min, double tail_div,
                  int tail_max = 6)
{
    P.pieces.clear();
    P.cta_off.assign(1, 0);
    const int UT = P.total_units, SL = (UT + nw - 1) / nw;
    const int min_st = std::max(tail_min, (2 * P.nbk + sub) / nw + 1);   // a piece must get past its own warm-up
    const long long total = (long long)P.npanels * SL;
    int panel = 0, ua = 0;
    auto take = [&](int st, int slack) {   // append the next piece of st stages (up to st + slack if that ends the line)
        const int ua0 = std::max(ua - P.nbk, 0) / sub * sub;   // stages start on a load-tile boundary
        const int rest = (UT - ua0 + nw - 1) / nw;
        int ub = UT, nst = rest;
        if (rest > st + slack) {
            ub = ua0 + st * nw - P.nbk;
            nst = st;
        }
        P.pieces.push_back(Piece{panel, ua, ub, nst});
        ua = ub;
        if (ua >= UT) { ++panel; ua = 0; }
        return nst;
    };
    const int quota = fixed > 0 ? 0 : (int)(static_frac * (double)total / slots);
    if (quota >= 2 * min_st && total >= 4LL * slots) {
        for (int c = 0; c < slots && panel < P.npanels; ++c) {
            int left = quota;
            while (left >= min_st && panel < P.npanels) left -= take(left, 1);
            P.cta_off.push_back((int)P.pieces.size());
        }
    }
    P.nstatic = (int)P.pieces.size();
    if (fixed == 0 && P.nstatic == 0 && total < 4LL * slots) {
        // Small problem (a CTA gets at most a few stages): one wave of equal pieces, at most one per CTA, because a
        // second piece on some CTAs would double the kernel time.  k pieces per line, each st stages.
        const int min_one = std::max(2, (2 * P.nbk + sub) / nw + 1);   // (tail_min is about the drawn tail only)
        const int k = (int)std::max<long long>(1, std::min<long long>(slots / P.npanels, SL / min_one));
        const int st = std::max(min_one, (UT + (k - 1) * 2 * P.nbk + k * nw - 1) / (k * nw));
        while (panel < P.npanels) take(st, st - 1);
        P.nstatic = (int)P.pieces.size();   // all static (CTA c owns pieces c, c + slots, ...: here just piece c):
        const int per = (P.nstatic + slots - 1) / slots;   // no ticket is ever drawn
        for (int c = 1; c <= slots; ++c) P.cta_off.push_back(std::min(P.nstatic, c * per));
        return;
    }
    double remaining = 0.0;
    if (panel < P.npanels) remaining = (double)(P.npanels - panel) * SL - (double)ua / nw;
    while (panel < P.npanels) {
        int st = fixed > 0 ? fixed : std::min(tail_max, (int)(remaining / (tail_div * slots)));
        st = std::max(st, min_st);
        const int ua_before = ua, panel_before = panel;
        take(st, (st + 1) / 2);
        const Piece& pc = P.pieces.back();
        (void)ua_before; (void)panel_before;
        remaining -= (double)(pc.ub - pc.ua) / nw;
    }
    while ((int)P.cta_off.size() < slots + 1) P.cta_off.push_back(P.nstatic);   // CTAs without a static share
}

// Early start (kernels.cuh): a static piece of direction d is "safe" if everything it reads and writes lies in grid
// lines that the OTHER direction's sweep completes within its static part, i.e. before the first panel that has a
// drawn piece.  Positions along a line of d are line indices of the other direction.  Each CTA's share is reordered
// safe-first, so that a CTA that becomes resident during the previous sweep's tail has something to do.
// Hazards: a safe piece writes only safe lines of a buffer in which the previous sweep's tail still reads at most its
// own (unsafe) lines -- scheme 0: w_{n+2} overwrites w_{n-1}; scheme 1: U^{k+1} overwrites V^{k-1}, V^{k+2} overwrites U^k,
// which the y sweep before it never touches.
void mark_safe_pieces(wave2d_t* h)
{
    for (int d = 0; d < 2; ++d) {
        DirPlan& P = h->plan[d];
        const DirPlan& O = h->plan[1 - d];
        for (Piece& pc : P.pieces) pc.safe = 0;
        P.has_safe = false;
        if (!h->opt_early || P.solver != WAVE2D_SOLVER_STREAM || O.solver != WAVE2D_SOLVER_STREAM ||
            P.nstatic == 0 || O.nstatic == 0 || O.nstatic >= (int)O.pieces.size())
            continue;
        const long long limit = (long long)O.pieces[O.nstatic].panel * 32 * O.var->vec;   // first line not surely done
        const Variant& V = *P.var;
        for (int i = 0; i < P.nstatic; ++i) {
            Piece& pc = P.pieces[i];
            const int gbase = std::max(pc.ua - P.nbk, 0) / V.sub * V.sub;
            const long long end = (long long)(gbase + pc.nst * V.nw) * V.unit + 16;   // + neighbour points, margin
            pc.safe = end <= limit ? 1 : 0;
            P.has_safe = P.has_safe || pc.safe != 0;
        }
        for (size_t c = 0; c + 1 < P.cta_off.size(); ++c)   // safe pieces first within a CTA's share
            std::stable_partition(P.pieces.begin() + P.cta_off[c], P.pieces.begin() + P.cta_off[c + 1],
                                  [](const Piece& q) { return q.safe != 0; });
    }
}

// x sweep load map: the field seen as (128-byte tile row, grid row, tile index along the row); a box of
// [ntiles][32 rows][128 B] lands in shared memory tile after tile, each 128B-swizzled, and is 32 rows x
// ntiles * 128 contiguous bytes in global memory.  Elements beyond n1 inside the last tile are the zero pad columns.
int make_tmap_x3(wave2d_t* h, CUtensorMap* tm, void* base, int ntiles)
{
    EncodeTiledFn enc = encode_tiled();
    if (!enc) {
        h->err = "cuTensorMapEncodeTiled entry point not available";
        return WAVE2D_ERR_CUDA;
    }
    const int tu = 128 / h->elem;
    const cuuint64_t dims[3] = {(cuuint64_t)tu, (cuuint64_t)h->n2, (cuuint64_t)(h->pitch / tu)};
    const cuuint64_t strides[2] = {(cuuint64_t)h->pitch * h->elem, 128};
    const cuuint32_t box[3] = {(cuuint32_t)tu, 32, (cuuint32_t)ntiles};
    const cuuint32_t es[3] = {1, 1, 1};
    CUresult r = enc(tm, h->dtype == WAVE2D_F64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3,
                     base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        char msg[160];
        snprintf(msg, sizeof msg, "cuTensorMapEncodeTiled (x sweep 3D map) failed (%d) n=%dx%d pitch=%lld", (int)r, h->n1,
                 h->n2, h->pitch);
        h->err = msg;
        return WAVE2D_ERR_CUDA;
    }
    return WAVE2D_OK;
}

// Exact path (exact.cuh): a group of wpc warps per line, segments of wpc * 32 * 8 points.
//   x: rows; nseg > 1 parks y of the whole line in shared memory (needs the full CTA per line).
//   y: strips of sc columns, the widest that fits the shared-memory budget, all rows of the strip on chip.
int plan_exact(wave2d_t* h, int d)
{
    DirPlan& P = h->plan[d];
    const int units = (P.n + EX_U - 1) / EX_U;
    int wpc = 1;
    while (wpc < EX_NW && wpc * 32 < units) wpc *= 2;        // power of two, so that it divides EX_NW
    const int nseg = (units + wpc * 32 - 1) / (wpc * 32);
    const bool var = h->have_cs;
    if (var && nseg > 1) {
        h->err = "variable speed: lines of more than 4096 unknowns are not supported yet";
        return WAVE2D_ERR_UNSUPPORTED;
    }
    const size_t budget = (var ? 224 : 200) * 1024;
    P.ex_wpc = wpc;
    if (d == 0) {
        P.ex_nseg = nseg;
        P.ex_sc = 0;
        // nseg > 1: the parked line; else the two prefetch slots of (2 NV + 1) 16-byte cells per thread (3 NV + 1 with cs)
        const size_t smem = nseg > 1 ? (size_t)nseg * wpc * 32 * EX_U * h->elem
                                     : (size_t)2 * ((var ? 3 : 2) * (EX_U * h->elem / 16) + 1) * EX_NT * 16;
        if (smem > budget) {
            const int seg = wpc * 32 * EX_U;   // a line is parked in whole segments
            char msg[160];
            snprintf(msg, sizeof msg, "exact solver: an x line of more than %d %s unknowns does not fit shared memory",
                     (int)(budget / ((size_t)seg * h->elem)) * seg, h->elem == 8 ? "fp64" : "fp32");
            h->err = msg;
            return WAVE2D_ERR_UNSUPPORTED;
        }
        P.ex_smem = (int)smem;
        const bool f64 = h->dtype == WAVE2D_F64;
        if (var) P.ex_fn = f64 ? reinterpret_cast<const void*>(&wave2d_exact_x<double, true, true>)
                               : reinterpret_cast<const void*>(&wave2d_exact_x<float, true, true>);
        else if (nseg == 1) P.ex_fn = f64 ? reinterpret_cast<const void*>(&wave2d_exact_x<double, false, true>)
                                          : reinterpret_cast<const void*>(&wave2d_exact_x<float, false, true>);
        else P.ex_fn = f64 ? reinterpret_cast<const void*>(&wave2d_exact_x<double, false, false>)
                           : reinterpret_cast<const void*>(&wave2d_exact_x<float, false, false>);
        const int passes = (P.nlines + EX_NW / wpc - 1) / (EX_NW / wpc);
        P.grid = passes;
    } else {
        const size_t col = (size_t)ex_cpitch(units) * h->elem * (var ? 2 : 1);   // one column of the strip (+ its a_p)
        int sc = 16;
        while (sc > 1 && sc * col > budget) sc /= 2;
        if (sc * col > budget) {
            int mu = (int)(budget / h->elem / (EX_U + 1));   // most units whose one-column strip still fits
            while (mu > 0 && (size_t)ex_cpitch(mu) * h->elem > budget) --mu;
            char msg[160];
            snprintf(msg, sizeof msg, "exact solver: a y line of more than %d %s unknowns does not fit shared memory",
                     mu * EX_U, h->elem == 8 ? "fp64" : "fp32");
            h->err = msg;
            return WAVE2D_ERR_UNSUPPORTED;
        }
        while (sc > 1 && (P.nlines + sc - 1) / sc < h->num_sms) sc /= 2;   // small grids: more, narrower strips
        P.ex_sc = sc;
        P.ex_nseg = nseg;
        P.ex_smem = (int)(sc * col);
        const bool f64 = h->dtype == WAVE2D_F64;
        if (var) P.ex_fn = f64 ? reinterpret_cast<const void*>(&wave2d_exact_y<double, true, true>)
                               : reinterpret_cast<const void*>(&wave2d_exact_y<float, true, true>);
        else if (nseg == 1) P.ex_fn = f64 ? reinterpret_cast<const void*>(&wave2d_exact_y<double, false, true>)
                                          : reinterpret_cast<const void*>(&wave2d_exact_y<float, false, true>);
        else P.ex_fn = f64 ? reinterpret_cast<const void*>(&wave2d_exact_y<double, false, false>)
                           : reinterpret_cast<const void*>(&wave2d_exact_y<float, false, false>);
        const int strips = (P.nlines + sc - 1) / sc;
        P.grid = strips;
    }
    W2D_CUDA(h, cudaFuncSetAttribute(P.ex_fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)budget));
    // persistent CTAs, one wave: a CTA's start-up (scalars, first loads) is paid once per SM slot, not once per few lines
    int per_sm = 0;
    W2D_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, P.ex_fn, EX_NT, (size_t)P.ex_smem));
    P.grid = std::max(1, std::min(P.grid, std::max(1, per_sm) * h->num_sms));
    return WAVE2D_OK;
}

int plan_dir(wave2d_t* h, int d)
{
    DirPlan& P = h->plan[d];
    P = DirPlan();
    P.n = d == 0 ? h->n1 : h->n2;
    P.nlines = d == 0 ? h->n2 : h->n1;
    P.shape = h->opt_shape[d];
    const int one = h->scheme == 1 && d == 1;
    if (one) {
        P.shape = std::min(P.shape, 1);
        // Large grids (>= 128 stages of 4096 points per SM): 16-point units halve the barrier rounds per point and
        // the longer pieces cost nothing there (config 5: +4.5 %); smaller grids keep 8-point units (shorter tail).
        const long long work = (long long)((P.nlines + 31) / 32) * ((P.n + 127) / 128);
        if (h->opt_shape[d] == 0 && h->elem == 8 && work >= 128LL * h->num_sms) P.shape = 1;
    }
    P.var = find_variant(h->elem, d, P.shape, one);
    if (P.var && P.var->vec == 2 && ((h->have_src && !one) || (h->pitch & 1))) P.var = find_variant(h->elem, d, P.shape + 1, one);
    if (!P.var) {
        h->err = "no kernel variant for this shape index";
        return WAVE2D_ERR_ARG;
    }
    const Variant& V = *P.var;
    const int U = V.unit;
    const double tol = h->dtype == WAVE2D_F64 ? 1e-17 : 1e-8;   // rho^H <= tol: below half an ulp of T
    const double tolp = h->dtype == WAVE2D_F64 ? 2e-15 : 1e-8;  // pivots count as stationary within a few ulp
    double rho = 0.0;
    int pconv = 0;   // rows [pconv, n) have stationary pivots (to tol) in every half-step
    for (int n = d; n < (h->table_period ? h->table_period : 2 * h->M); n += 2) {
        const double* row = &h->table[static_cast<size_t>(n) * ROW_DOUBLES];
        if (row[ROW_BETA] == 0.0) continue;   // unused row (scheme 1 has M - 1 steps)
        rho = std::max(rho, row[ROW_RHO]);
        int pc = KMAX + 1;
        for (int p = KMAX - 1; p >= 0 && std::fabs(row[ROW_CP + p] - row[ROW_RHO]) <= tolp * row[ROW_RHO] &&
                               std::fabs(row[ROW_INVP + p] - row[ROW_INV]) <= tolp * row[ROW_INV]; --p)
            pc = p;
        pconv = std::max(pconv, pc);
    }
    P.rho = rho;
    int H = 1;
    if (rho > 0.0) H = std::max(1, (int)std::ceil(std::log(tol) / std::log(rho)));
    P.halo = H;
    const int nbk = (H + U - 1) / U;
    const bool fits = nbk <= std::min(NBK_MAX, V.nw) && pconv <= KMAX;
    if (h->have_cs && h->opt_solver == WAVE2D_SOLVER_STREAM) {
        h->err = "variable speed: the streamed kernels assume Toeplitz systems (use solver AUTO or EXACT)";
        return WAVE2D_ERR_UNSUPPORTED;
    }
    if (h->have_cs || h->opt_solver == WAVE2D_SOLVER_EXACT || (h->opt_solver == WAVE2D_SOLVER_AUTO && !fits)) {
        P.solver = WAVE2D_SOLVER_EXACT;
        return plan_exact(h, d);
    }
    if (!fits) {
        h->err = "streamed solver: decay bound rho^H <= tol needs a longer carry series than supported";
        return WAVE2D_ERR_UNSUPPORTED;
    }
    P.solver = WAVE2D_SOLVER_STREAM;
    P.nbk = nbk;
    P.halo = nbk * U;
    P.kb = (pconv + U - 1) / U;
    W2D_CUDA(h, cudaFuncSetAttribute(V.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, V.smem));
    if (V.fn_nosrc) W2D_CUDA(h, cudaFuncSetAttribute(V.fn_nosrc, cudaFuncAttributeMaxDynamicSharedMemorySize, V.smem));
    if (V.fn_dense) W2D_CUDA(h, cudaFuncSetAttribute(V.fn_dense, cudaFuncAttributeMaxDynamicSharedMemorySize, V.smem));
    int per_sm = 0;
    W2D_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, V.fn, V.threads, V.smem));
    if (per_sm < 1) {
        h->err = "sweep kernel does not fit on an SM";
        return WAVE2D_ERR_UNSUPPORTED;
    }
    P.ctas_per_sm = per_sm;
    P.npanels = ((P.nlines + V.vec - 1) / V.vec + 31) / 32;   // 32 lanes, V.vec lines each
    P.total_units = (P.n + U - 1) / U;
    // Persistent grid, one wave; the CTAs draw the pieces from an atomic ticket counter.
    const int slots = per_sm * h->num_sms;
    // shortest drawn piece: ~16 K points of work per line panel (4 stages of 4096 points in fp64, 2 of 8192 in fp32):
    // shorter pieces pay relatively more for their carry warm-up, longer ones lengthen the tail of the kernel
    const int stage_points = V.nw * V.unit * 32 * V.vec;
    const int tail_min = h->opt_tail_min > 0 ? h->opt_tail_min : std::min(6, std::max(2, 16384 / stage_points));
    // share dealt out statically: 0.70 in fp64, 0.75 in fp32.  The effect is a step function of the resulting quota of
    // stages per CTA and depends on how the shares fall on the line ends (r2 sweeps, reproducible to 0.1 us): 4095^2 fp64
    // quota 18 / 19 / 20 / 21 -> 129.1 / 128.4 / 130.0 / 131.4 us per step, 8191 x 2047 fp64 129.5 / 130.2 / 127.4 / 128.6;
    // fp32 loses 1-2 % below 0.75.  0.70 takes the quota of the configuration the roofline target is quoted on.
    const double static_frac = h->opt_static_frac >= 0.0 ? h->opt_static_frac : h->elem == 8 ? 0.70 : 0.75;
    build_pieces(P, V.nw, V.sub, slots, h->opt_quota[d], static_frac, tail_min, h->opt_tail_div,
                 h->opt_tail_max);
    P.quota = h->opt_quota[d];
    P.grid = slots;
    return WAVE2D_OK;
}

int build_graphs(wave2d_t* h);

// ---- small grids: one cluster, one launch for the whole step loop (line.cuh) --------------------------------
constexpr int LINE_WARPS = 16;   // warps per CTA of the small-grid kernel

template <typename T, int U>
const void* line_kernel() { return reinterpret_cast<const void*>(&wave2d_line_steps<T, U, LINE_WARPS>); }
template <typename T, int U>
const void* resident_kernel() { return reinterpret_cast<const void*>(&wave2d_line_resident<T, U, LINE_WARPS>); }

int plan_line(wave2d_t* h)
{
    h->line_mode = false;
    const int nmax = std::max(h->n1, h->n2);
    const bool fits = nmax <= 32 * 8;
    if (h->opt_solver == WAVE2D_SOLVER_LINE && !fits) {
        h->err = "solver LINE: more than 256 unknowns per line";
        return WAVE2D_ERR_UNSUPPORTED;
    }
    if (h->have_cs && h->opt_solver == WAVE2D_SOLVER_LINE) {
        h->err = "variable speed: the small-grid kernel assumes Toeplitz systems (use solver AUTO or EXACT)";
        return WAVE2D_ERR_UNSUPPORTED;
    }
    if (!fits || h->have_cs || (h->opt_solver != WAVE2D_SOLVER_AUTO && h->opt_solver != WAVE2D_SOLVER_LINE)) return WAVE2D_OK;
    const int U = nmax <= 32 * 4 ? 4 : 8;
    h->line_unit = U;
    if (h->dtype == WAVE2D_F64) h->line_fn = U == 4 ? line_kernel<double, 4>() : line_kernel<double, 8>();
    else h->line_fn = U == 4 ? line_kernel<float, 4>() : line_kernel<float, 8>();
    h->line_smem = 2 * 16 * (32 * U + 1) * h->elem;
    // one CTA per 16 rows of the x half-step / per 16-column strip of the y half-step, at most one portable cluster
    const int want = std::max((h->n2 + LINE_WARPS - 1) / LINE_WARPS, (h->n1 + 15) / 16);
    h->line_ctas = std::max(1, std::min(8, want));
    // Split scheme, six line buffers per CTA within shared memory: the fields stay on chip for the whole launch
    h->line_resident = false;
    if (h->scheme == 0 && h->opt_resident) {
        const int lb = std::max((h->n2 + h->line_ctas - 1) / h->line_ctas, (h->n1 + h->line_ctas - 1) / h->line_ctas);
        const size_t need = (size_t)6 * lb * (32 * U + 1) * h->elem;
        if (need <= 200 * 1024) {
            h->line_resident = true;
            h->line_smem = (int)need;
            if (h->dtype == WAVE2D_F64) h->line_fn = U == 4 ? resident_kernel<double, 4>() : resident_kernel<double, 8>();
            else h->line_fn = U == 4 ? resident_kernel<float, 4>() : resident_kernel<float, 8>();
        }
    }
    W2D_CUDA(h, cudaFuncSetAttribute(h->line_fn, cudaFuncAttributeMaxDynamicSharedMemorySize, h->line_smem));
    for (int d = 0; d < 2; ++d) {
        DirPlan& P = h->plan[d];
        P = DirPlan();
        P.solver = WAVE2D_SOLVER_LINE;
        P.n = d == 0 ? h->n1 : h->n2;
        P.nlines = d == 0 ? h->n2 : h->n1;
        P.grid = h->line_ctas;
        for (int n = d; n < (h->table_period ? h->table_period : 2 * h->M); n += 2)
            P.rho = std::max(P.rho, h->table[static_cast<size_t>(n) * ROW_DOUBLES + ROW_RHO]);
    }
    h->line_mode = true;
    return WAVE2D_OK;
}

// All `steps` time steps in one launch (the kernel advances the device step counter itself).
int launch_line_steps(wave2d_t* h, int steps)
{
    LineArgs a;
    a.table = h->d_table; a.table_period = h->table_period; a.d_k = h->d_k; a.nsteps = steps;
    a.ring = h->scheme == 1 ? 4 : 3; a.one_y = h->scheme == 1 ? 1 : 0;
    for (int b = 0; b < 4; ++b) a.bufs[b] = h->buf[b];
    a.n1 = h->n1; a.n2 = h->n2; a.pitch = h->pitch;
    a.src[0] = h->have_src ? h->src_dev[0] : nullptr;
    a.src[1] = h->have_src && h->scheme == 0 ? h->src_dev[1] : nullptr;   // scheme 1: f enters in x only
    a.win_i0 = h->win_i0; a.win_j0 = h->win_j0; a.win_w = h->win_w; a.win_h = h->win_h;
    a.g2 = h->scheme == 1 ? 2.0 : 2.0 * h->gamma;
    void* args[1] = {&a};
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(h->line_ctas);
    cfg.blockDim = dim3(32 * LINE_WARPS);
    cfg.dynamicSmemBytes = h->line_smem;
    cfg.stream = h->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = h->line_ctas;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    W2D_CUDA(h, cudaLaunchKernelExC(&cfg, h->line_fn, args));
    h->launches += 1;
    h->line_launches += 1;
    return WAVE2D_OK;
}

int ensure_plan(wave2d_t* h)
{
    if (h->plan_ok) return WAVE2D_OK;
    drop_graph(h);
    build_table(h);
    dev_free(h, h->d_table, h->table_bytes);
    h->d_table = nullptr;
    const size_t tbytes = h->table.size() * sizeof(double);
    if (tbytes > (size_t)1 << 30) {
        h->err = "per-half-step table would exceed 1 GiB (M too large)";
        return WAVE2D_ERR_UNSUPPORTED;
    }
    int st = dev_alloc(h, reinterpret_cast<void**>(&h->d_table), tbytes);
    if (st) return st;
    h->table_bytes = tbytes;
    W2D_CUDA(h, cudaMemcpyAsync(h->d_table, h->table.data(), tbytes, cudaMemcpyHostToDevice, h->stream));
    W2D_CUDA(h, cudaStreamSynchronize(h->stream));
    st = plan_line(h);
    if (st) return st;
    if (h->line_mode) {
        h->plan_ok = true;
        return WAVE2D_OK;
    }
    for (int d = 0; d < 2; ++d) {
        st = plan_dir(h, d);
        if (st) return st;
    }
    mark_safe_pieces(h);
    memset(h->maps, 0, sizeof h->maps);
    for (int b = 0; b < (h->scheme == 1 ? 4 : 3); ++b) {
        if (h->plan[0].solver == WAVE2D_SOLVER_STREAM) {
            const int U = h->plan[0].var->unit;
            st = make_tmap_x3(h, &h->maps[0].load[b], h->buf[b], h->plan[0].var->nw / h->plan[0].var->sub);
            if (st == WAVE2D_OK) st = make_tmap(h, &h->maps[0].store[b], h->buf[b], U, 32, U * h->elem);   // one warp's unit
            if (st == WAVE2D_OK) st = make_tmap(h, &h->maps[0].edge[b], h->buf[b], 16 / h->elem, 32, 0);
            if (st) return st;
        }
        if (h->plan[1].solver == WAVE2D_SOLVER_STREAM) {
            const Variant& V = *h->plan[1].var;
            st = make_tmap(h, &h->maps[1].load[b], h->buf[b], 32 * V.vec, V.unit * V.nw + (V.one ? 0 : 2), 0);
            if (st) return st;
        }
    }
    for (int d = 0; d < 2; ++d) {
        dev_free(h, h->d_pieces[d], h->pieces_bytes[d]);
        dev_free(h, h->d_cta_off[d], h->cta_off_bytes[d]);
        dev_free(h, h->d_trace[d], h->trace_bytes[d]);
        h->d_pieces[d] = nullptr;
        h->d_cta_off[d] = nullptr;
        h->d_trace[d] = nullptr;
        const DirPlan& P = h->plan[d];
        if (P.solver != WAVE2D_SOLVER_STREAM) continue;
        const size_t pb = std::max<size_t>(1, P.pieces.size()) * sizeof(Piece), ob = P.cta_off.size() * sizeof(int);
        st = dev_alloc(h, reinterpret_cast<void**>(&h->d_pieces[d]), pb);
        if (st) return st;
        h->pieces_bytes[d] = pb;
        st = dev_alloc(h, reinterpret_cast<void**>(&h->d_cta_off[d]), ob);
        if (st) return st;
        h->cta_off_bytes[d] = ob;
        W2D_CUDA(h, cudaMemcpy(h->d_cta_off[d], P.cta_off.data(), ob, cudaMemcpyHostToDevice));
        if (!P.pieces.empty())
            W2D_CUDA(h, cudaMemcpy(h->d_pieces[d], P.pieces.data(), P.pieces.size() * sizeof(Piece), cudaMemcpyHostToDevice));
        if (h->opt_trace) {
            const size_t tb = (size_t)P.grid * 16 * sizeof(unsigned long long);
            st = dev_alloc(h, reinterpret_cast<void**>(&h->d_trace[d]), tb);
            if (st) return st;
            h->trace_bytes[d] = tb;
            W2D_CUDA(h, cudaMemset(h->d_trace[d], 0, tb));
        }
    }
    h->plan_ok = true;
    // The step loop's graphs are part of the plan: captured, instantiated and uploaded here, never inside a run call
    // that may be timed (wave2d_run(h, 0) forces the plan).
    if (h->opt_graph) {
        st = build_graphs(h);
        if (st) {
            h->plan_ok = false;
            return st;
        }
    }
    return WAVE2D_OK;
}

FieldSet field_set(const wave2d_t* h)
{
    FieldSet fs;
    for (int b = 0; b < 4; ++b) fs.b[b] = h->buf[b];
    fs.ring = h->scheme == 1 ? 4 : 3;
    return fs;
}

// Arguments of a whole-line half-step (exact.cuh) of direction d that do not depend on the time level.
ExactArgs exact_args(const wave2d_t* h, int d)
{
    const DirPlan& P = h->plan[d];
    ExactArgs a = {};
    a.fs = field_set(h);
    a.table = h->d_table; a.period = h->table_period;
    a.n = P.n; a.nlines = P.nlines; a.pitch = h->pitch;
    a.src = h->have_src && !(h->scheme == 1 && d == 1) ? h->src_dev[d] : nullptr;   // scheme 1: f enters in x only
    a.sl0 = d == 0 ? h->win_j0 : h->win_i0; a.snl = d == 0 ? h->win_h : h->win_w;
    a.sp0 = d == 0 ? h->win_i0 : h->win_j0; a.snp = d == 0 ? h->win_w : h->win_h;
    a.g2 = h->scheme == 1 ? 2.0 : 2.0 * h->gamma;
    a.one = h->scheme == 1 && d == 1;
    a.wpc = P.ex_wpc; a.nseg = P.ex_nseg; a.sc = P.ex_sc;
    a.cs = h->d_cs;
    a.gamma = h->gamma;
    return a;
}

// One half-step: sweep n_off of the current chunk (the kernels add twice the device step counter; the direction is
// the parity of n_off, the buffer roles follow on the device).  after_own: the previous kernel on `stream` is sweep
// n_off - 1 of this chunk, so this one may be chained to it by programmatic dependent launch (and start early).
int launch_half_step(wave2d_t* h, cudaStream_t stream, int n_off, bool after_own)
{
    const int d = n_off & 1;
    Range range(d == 0 ? "x_sweep" : "y_sweep");   // (launch or capture of the sweep; a graph replay is inside "wave2d_run")
    const DirPlan& P = h->plan[d];
    const int* dk = h->d_k;
    const void* src = h->have_src && !(h->scheme == 1 && d == 1) ? h->src_dev[d] : nullptr;   // scheme 1: f enters in x only
    const int sl0 = d == 0 ? h->win_j0 : h->win_i0, snl = d == 0 ? h->win_h : h->win_w;
    const int sp0 = d == 0 ? h->win_i0 : h->win_j0, snp = d == 0 ? h->win_w : h->win_h;
    if (P.solver == WAVE2D_SOLVER_STREAM) {
        SweepArgs a;
        a.table = h->d_table; a.table_period = h->table_period; a.d_k = dk; a.n_off = n_off;
        a.ring = h->scheme == 1 ? 4 : 3;
        for (int b = 0; b < 4; ++b) a.bufs[b] = h->buf[b];
        a.n = P.n; a.nlines = (P.nlines + P.var->vec - 1) / P.var->vec; a.nbk = P.nbk; a.kb = P.kb;
        a.pieces = h->d_pieces[d]; a.npieces = (int)P.pieces.size(); a.tickets = h->d_tickets;
        a.done = h->d_tickets + SLOTS;
        a.early = h->opt_early && h->opt_pdl && after_own && h->plan[1 - d].solver == WAVE2D_SOLVER_STREAM;
        a.prev_grid = h->plan[1 - d].grid;
        a.signal = h->plan[1 - d].has_safe ? 1 : 0;
        a.cta_off = h->d_cta_off[d]; a.nstatic = P.nstatic;
        a.pitch = h->pitch / P.var->vec;   // in units of the kernel's T
        a.src = src; a.sl0 = sl0; a.snl = snl; a.sp0 = sp0; a.snp = snp;
        a.g2 = h->scheme == 1 ? 2.0 : 2.0 * h->gamma;
        a.trace = h->opt_trace ? h->d_trace[d] : nullptr;
        void* args[2] = {&h->maps[d], &a};
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(P.grid);
        cfg.blockDim = dim3(P.var->threads);
        cfg.dynamicSmemBytes = P.var->smem;
        cfg.stream = stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // overlap our prologue with the previous
        at[0].val.programmaticStreamSerializationAllowed = 1;            // kernel's tail (griddepcontrol.wait inside)
        cfg.attrs = at;
        // Only behind a sweep of the same chunk: the first sweep of a chunk follows wave2d_end_chunk (or a copy) and
        // reads the step counter before griddepcontrol.wait, so it must see it final.
        cfg.numAttrs = h->opt_pdl && after_own ? 1 : 0;
        // a window that covers more than 1/8 of the grid counts as dense (kernels.cuh, SRCM)
        const bool dense = src != nullptr && 8.0 * h->win_w * h->win_h > (double)h->n1 * h->n2;
        const void* fn = src == nullptr && P.var->fn_nosrc ? P.var->fn_nosrc : dense && P.var->fn_dense ? P.var->fn_dense : P.var->fn;
        W2D_CUDA(h, cudaLaunchKernelExC(&cfg, fn, args));
        return WAVE2D_OK;
    }
    // exact path: the whole-line solver of the direction (exact.cuh)
    ExactArgs a = exact_args(h, d);
    a.d_k = dk; a.n_off = n_off;
    void* args[1] = {&a};
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(P.grid);
    cfg.blockDim = dim3(EX_NT);
    cfg.dynamicSmemBytes = P.ex_smem;
    cfg.stream = stream;
    W2D_CUDA(h, cudaLaunchKernelExC(&cfg, P.ex_fn, args));
    return WAVE2D_OK;
}

int kernels_per_sweep(const wave2d_t* h, int d)
{
    (void)h; (void)d;
    return 1;
}

// A chunk of the step loop (A7): `steps` time steps = sweeps n_off = 0 .. 2 steps - 1 relative to the device step
// counter, then wave2d_end_chunk, which counts them and re-zeroes the counters they used.  The same sequence is
// either captured into a graph (once, with the plan) or launched directly (option graph = 0).
int launch_chunk(wave2d_t* h, cudaStream_t stream, int steps)
{
    int st = WAVE2D_OK;
    for (int s = 0; s < steps && st == WAVE2D_OK; ++s) {
        st = launch_half_step(h, stream, 2 * s, s > 0 && h->plan[1].solver == WAVE2D_SOLVER_STREAM);
        if (st == WAVE2D_OK) st = launch_half_step(h, stream, 2 * s + 1, h->plan[0].solver == WAVE2D_SOLVER_STREAM);
    }
    if (st) return st;
    wave2d_end_chunk<<<1, 2 * SLOTS, 0, stream>>>(h->d_k, steps, h->d_tickets);
    W2D_CUDA(h, cudaGetLastError());
    return WAVE2D_OK;
}

long long kernels_per_chunk(const wave2d_t* h, int steps)
{
    return (long long)steps * (kernels_per_sweep(h, 0) + kernels_per_sweep(h, 1)) + 1;
}

// Graphs of 1, 2, 4, ... opt_graph_steps time steps: any step count is a short sequence of replays, at any phase of
// the buffer ring (the kernels derive the roles from the device step counter), with no plain launch left over.
// Captured on the handle's own stream (capture needs a non-legacy stream; the executables launch into any stream).
int build_graphs(wave2d_t* h)
{
    drop_graph(h);
    for (int i = 0; i < NCHUNK && (1 << i) <= h->opt_graph_steps; ++i) {
        cudaGraph_t g = nullptr;
        W2D_CUDA(h, cudaStreamBeginCapture(h->own_stream, cudaStreamCaptureModeThreadLocal));
        const int st = launch_chunk(h, h->own_stream, 1 << i);
        const cudaError_t e = cudaStreamEndCapture(h->own_stream, &g);
        if (st != WAVE2D_OK) {
            if (g) cudaGraphDestroy(g);
            (void)cudaGetLastError();
            return st;
        }
        if (e != cudaSuccess) {
            h->err = std::string("cudaStreamEndCapture: ") + cudaGetErrorString(e);
            (void)cudaGetLastError();
            return WAVE2D_ERR_CUDA;
        }
        const cudaError_t ei = cudaGraphInstantiate(&h->gexec[i], g, 0);
        cudaGraphDestroy(g);
        if (ei != cudaSuccess) {
            h->gexec[i] = nullptr;
            h->err = std::string("cudaGraphInstantiate: ") + cudaGetErrorString(ei);
            (void)cudaGetLastError();
            return WAVE2D_ERR_CUDA;
        }
        W2D_CUDA(h, cudaGraphUpload(h->gexec[i], h->own_stream));   // first replay pays no upload
    }
    W2D_CUDA(h, cudaStreamSynchronize(h->own_stream));
    return WAVE2D_OK;
}

int copy_in(wave2d_t* h, void* dst, const void* src, long ld)
{
    W2D_CUDA(h, cudaMemcpy2DAsync(dst, (size_t)h->pitch * h->elem, src, (size_t)ld * h->elem, (size_t)h->n1 * h->elem,
                                  h->n2, cudaMemcpyDefault, h->stream));
    return WAVE2D_OK;
}

int copy_out(wave2d_t* h, void* dst, long ld, const void* src)
{
    if (!h || !dst || ld < h->n1) return WAVE2D_ERR_ARG;
    if (!h->have_initial) return WAVE2D_ERR_STATE;
    W2D_CUDA(h, cudaMemcpy2DAsync(dst, (size_t)ld * h->elem, src, (size_t)h->pitch * h->elem, (size_t)h->n1 * h->elem,
                                  h->n2, cudaMemcpyDefault, h->stream));
    W2D_CUDA(h, cudaStreamSynchronize(h->stream));
    return WAVE2D_OK;
}


// Scheme 1 start, (2.9) as printed: U^0 = phi -> buf[3], U^1 = phi + tau psi -> buf[0]; the state
// is time level k = 1.  V^0, V^1 follow at the first run (they need the final speed samples).
int set_initial_factored(wave2d_t* h, const void* phi, const void* psi, long ld)
{
    if (h->M < 1) return WAVE2D_ERR_RANGE;
    int st = copy_in(h, h->buf[3], phi, ld);
    if (st == WAVE2D_OK && psi) st = copy_in(h, h->buf[2], psi, ld);
    if (st) return st;
    const dim3 blk(128), grd((h->n1 + 127) / 128, h->n2);
    if (h->dtype == WAVE2D_F64)
        wave2d_init_prev<double><<<grd, blk, 0, h->stream>>>((double*)h->buf[0], (const double*)h->buf[3],
                                                             psi ? (const double*)h->buf[2] : nullptr, h->n1, h->n2,
                                                             h->pitch, -h->tau);
    else
        wave2d_init_prev<float><<<grd, blk, 0, h->stream>>>((float*)h->buf[0], (const float*)h->buf[3],
                                                            psi ? (const float*)h->buf[2] : nullptr, h->n1, h->n2,
                                                            h->pitch, -h->tau);
    W2D_CUDA(h, cudaGetLastError());
    W2D_CUDA(h, cudaMemsetAsync(h->d_k, 0, sizeof(int), h->stream));
    W2D_CUDA(h, cudaMemsetAsync(h->d_tickets, 0, (size_t)2 * SLOTS * sizeof(int), h->stream));
    W2D_CUDA(h, cudaStreamSynchronize(h->stream));
    h->have_initial = true;
    h->v_ready = false;
    h->k = 1;
    h->ran = false;
    return WAVE2D_OK;
}

// Scheme 1: V^0 = (I - ay(c^0) Dy) U^0 -> buf[1], V^1 = (I - ay(c^1) Dy) U^1 -> buf[2]   (roles of solve t = 0)
int init_factored_v(wave2d_t* h)
{
    if (h->opt_start == 2) {   // U^1 += tau^2 / 2 (c^0 Lap_h phi + g^0 s): U^0 = phi in buf[3], U^1 in buf[0]
        const double h1 = h->l / h->N1, hy = step_y(h), ht2 = 0.5 * h->tau * h->tau;
        const double g0 = h->have_src ? (h->g_half.empty() ? 1.0 : h->g_half[0]) : 0.0;
        const dim3 blk(128), grd((h->n1 + 127) / 128, h->n2);
        if (h->dtype == WAVE2D_F64)
            wave2d_start2<double><<<grd, blk, 0, h->stream>>>((double*)h->buf[0], (const double*)h->buf[3], h->n1, h->n2, h->pitch,
                                                              ht2 * h->c_half[0] / (h1 * h1), ht2 * h->c_half[0] / (hy * hy), ht2 * g0,
                                                              (const double*)h->src_dev[1], h->win_i0, h->win_j0, h->win_w, h->win_h);
        else
            wave2d_start2<float><<<grd, blk, 0, h->stream>>>((float*)h->buf[0], (const float*)h->buf[3], h->n1, h->n2, h->pitch,
                                                             ht2 * h->c_half[0] / (h1 * h1), ht2 * h->c_half[0] / (hy * hy), ht2 * g0,
                                                             (const float*)h->src_dev[1], h->win_i0, h->win_j0, h->win_w, h->win_h);
        W2D_CUDA(h, cudaGetLastError());
        h->launches += 1;
    }
    const double h2 = step_y(h), t2 = h->tau * h->tau;
    const double ay0 = t2 * h->c_half[0] / (2.0 * h2 * h2), ay1 = t2 * h->c_half[2] / (2.0 * h2 * h2);
    const dim3 blk(128), grd((h->n1 + 127) / 128, h->n2);
    if (h->dtype == WAVE2D_F64) {
        wave2d_apply_y<double><<<grd, blk, 0, h->stream>>>((double*)h->buf[1], (const double*)h->buf[3], h->n1, h->n2, h->pitch, ay0);
        wave2d_apply_y<double><<<grd, blk, 0, h->stream>>>((double*)h->buf[2], (const double*)h->buf[0], h->n1, h->n2, h->pitch, ay1);
    } else {
        wave2d_apply_y<float><<<grd, blk, 0, h->stream>>>((float*)h->buf[1], (const float*)h->buf[3], h->n1, h->n2, h->pitch, ay0);
        wave2d_apply_y<float><<<grd, blk, 0, h->stream>>>((float*)h->buf[2], (const float*)h->buf[0], h->n1, h->n2, h->pitch, ay1);
    }
    W2D_CUDA(h, cudaGetLastError());
    h->launches += 2;
    h->v_ready = true;
    return WAVE2D_OK;
}

}  // namespace

// =====================================================================================================
extern "C" {

int wave2d_create(wave2d_t** out, int N1, int N2, double l, double tau, int M, int dtype)
{
    if (!out) return WAVE2D_ERR_ARG;
    *out = nullptr;
    if (N1 < 2 || N2 < 2 || !(l > 0.0) || !(tau > 0.0) || M < 0 || (dtype != WAVE2D_F64 && dtype != WAVE2D_F32))
        return WAVE2D_ERR_ARG;
    wave2d_t* h = new (std::nothrow) wave2d_t();
    if (!h) return WAVE2D_ERR_ALLOC;
    h->N1 = N1; h->N2 = N2; h->n1 = N1 - 1; h->n2 = N2 - 1; h->M = M; h->dtype = dtype;
    h->elem = dtype == WAVE2D_F64 ? 8 : 4;
    h->l = l; h->tau = tau;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess || prop.major != 10) {
        (void)cudaGetLastError();
        delete h;
        return WAVE2D_ERR_CUDA;   // no device, or not an sm_100-class device: there is no other code path
    }
    h->num_sms = prop.multiProcessorCount;
    if (cudaStreamCreateWithFlags(&h->own_stream, cudaStreamNonBlocking) != cudaSuccess) {
        (void)cudaGetLastError();
        delete h;
        return WAVE2D_ERR_CUDA;
    }
    h->stream = h->own_stream;
    const int per128 = 128 / h->elem;
    h->pitch = ((long long)h->n1 + per128 - 1) / per128 * per128;     // rows start 128-byte aligned (H5)
    const size_t fbytes = (size_t)h->pitch * h->n2 * h->elem;
    int st = WAVE2D_OK;
    for (int b = 0; b < 3 && st == WAVE2D_OK; ++b) st = dev_alloc(h, &h->buf[b], fbytes);
    if (st == WAVE2D_OK) st = dev_alloc(h, reinterpret_cast<void**>(&h->d_k), sizeof(int));
    const size_t tk_bytes = (size_t)2 * SLOTS * sizeof(int);   // tickets[SLOTS] | done[SLOTS]
    if (st == WAVE2D_OK) st = dev_alloc(h, reinterpret_cast<void**>(&h->d_tickets), tk_bytes);
    if (st == WAVE2D_OK) {
        for (int b = 0; b < 3; ++b) cudaMemsetAsync(h->buf[b], 0, fbytes, h->stream);
        cudaMemsetAsync(h->d_k, 0, sizeof(int), h->stream);
        cudaMemsetAsync(h->d_tickets, 0, tk_bytes, h->stream);
        if (cudaStreamSynchronize(h->stream) != cudaSuccess) st = WAVE2D_ERR_CUDA;
    }
    if (st != WAVE2D_OK) {
        (void)cudaGetLastError();
        wave2d_destroy(h);
        return st;
    }
    h->c_half.assign((size_t)2 * M + 1, 1.0);
    *out = h;
    return WAVE2D_OK;
}

void wave2d_destroy(wave2d_t* h)
{
    if (!h) return;
    if (h->stream) cudaStreamSynchronize(h->stream);
    drop_graph(h);
    if (!h->ext_fields)
        for (int b = 0; b < 4; ++b) cudaFree(h->buf[b]);
    cudaFree(h->src_dev[0]);
    cudaFree(h->src_dev[1]);
    cudaFree(h->d_cs);
    cudaFree(h->d_table);
    cudaFree(h->d_k);
    for (int d = 0; d < 2; ++d) {
        cudaFree(h->d_pieces[d]);
        cudaFree(h->d_cta_off[d]);
        cudaFree(h->d_trace[d]);
    }
    cudaFree(h->d_tickets);
    if (h->own_stream) cudaStreamDestroy(h->own_stream);
    (void)cudaGetLastError();
    delete h;
}

int wave2d_set_stream(wave2d_t* h, void* cuda_stream)
{
    if (!h) return WAVE2D_ERR_ARG;
    W2D_CUDA(h, cudaStreamSynchronize(h->stream));
    h->stream = cuda_stream ? static_cast<cudaStream_t>(cuda_stream) : h->own_stream;
    return WAVE2D_OK;   // the graphs of the plan launch into any stream
}

int wave2d_set_option(wave2d_t* h, const char* name, double value)
{
    if (!h || !name) return WAVE2D_ERR_ARG;
    if (h->ran) return WAVE2D_ERR_STATE;
    const int iv = (int)value;
    if (!strcmp(name, "gamma")) { if (!(value > 0.0)) return WAVE2D_ERR_ARG; h->gamma = value; }
    else if (!strcmp(name, "kappa")) h->kappa = value;
    else if (!strcmp(name, "ly")) { if (!(value >= 0.0)) return WAVE2D_ERR_ARG; h->ly = value; }
    else if (!strcmp(name, "sigma")) {
        if (!(value > 0.0 && value <= 1.0)) return WAVE2D_ERR_ARG;
        if (h->scheme == 1 && value != 0.5) return WAVE2D_ERR_UNSUPPORTED;   // (2.8) has the weight 1/2 by definition
        h->sigma = value;
    }
    else if (!strcmp(name, "start")) {
        if (iv != 1 && iv != 2) return WAVE2D_ERR_ARG;
        h->opt_start = iv;
    }
    else if (!strcmp(name, "scheme")) {
        if ((iv != 0 && iv != 1) || h->have_initial) return WAVE2D_ERR_ARG;
        if (iv == 1 && (h->have_cs || h->sigma != 0.5)) return WAVE2D_ERR_UNSUPPORTED;   // variable speed, sigma: split scheme only
        if (iv == 1 && !h->buf[3]) {
            if (h->ext_fields) {   // a three-field workspace is attached: the scheme has to be chosen before it
                h->err = "scheme 1 needs a fourth field: set the scheme before wave2d_set_workspace";
                return WAVE2D_ERR_STATE;
            }
            const size_t fbytes = (size_t)h->pitch * h->n2 * h->elem;
            int st = dev_alloc(h, &h->buf[3], fbytes);
            if (st) return st;
            cudaMemsetAsync(h->buf[3], 0, fbytes, h->stream);
        }
        h->scheme = iv;
    }
    else if (!strcmp(name, "solver")) { if (iv < 0 || iv > 3) return WAVE2D_ERR_ARG; h->opt_solver = iv; }
    else if (!strcmp(name, "graph")) h->opt_graph = iv != 0;
    else if (!strcmp(name, "graph_steps")) {
        if (iv < 1 || iv > MAX_CHUNK || (iv & (iv - 1))) return WAVE2D_ERR_ARG;   // 1, 2, 4, ..., MAX_CHUNK
        h->opt_graph_steps = iv;
    }
    else if (!strcmp(name, "shape_x")) { if (iv < 0 || iv >= NVAR) return WAVE2D_ERR_ARG; h->opt_shape[0] = iv; }
    else if (!strcmp(name, "shape_y")) { if (iv < 0 || iv >= NVAR) return WAVE2D_ERR_ARG; h->opt_shape[1] = iv; }
    else if (!strcmp(name, "resident")) h->opt_resident = iv != 0;
    else if (!strcmp(name, "trace")) h->opt_trace = iv != 0;
    else if (!strcmp(name, "pdl")) h->opt_pdl = iv != 0;
    else if (!strcmp(name, "early")) h->opt_early = iv != 0;
    else if (!strcmp(name, "tail_max")) { if (iv < 1) return WAVE2D_ERR_ARG; h->opt_tail_max = iv; }
    else if (!strcmp(name, "tail_min")) { if (iv < 0) return WAVE2D_ERR_ARG; h->opt_tail_min = iv; }
    else if (!strcmp(name, "tail_div")) { if (!(value >= 0.25)) return WAVE2D_ERR_ARG; h->opt_tail_div = value; }
    else if (!strcmp(name, "static_frac")) { if (!(value >= 0.0 && value <= 1.0)) return WAVE2D_ERR_ARG; h->opt_static_frac = value; }
    else if (!strcmp(name, "quota_x")) { if (iv < 0) return WAVE2D_ERR_ARG; h->opt_quota[0] = iv; }
    else if (!strcmp(name, "quota_y")) { if (iv < 0) return WAVE2D_ERR_ARG; h->opt_quota[1] = iv; }
    else return WAVE2D_ERR_ARG;
    invalidate_plan(h);
    return WAVE2D_OK;
}

// bytes of one time level inside a caller's workspace (a multiple of 256, so that every level starts 256-byte aligned)
static size_t workspace_slice(const wave2d_t* h)
{
    return ((size_t)h->pitch * h->n2 * h->elem + 255) / 256 * 256;
}

int wave2d_workspace_bytes(const wave2d_t* h, unsigned long long* bytes)
{
    if (!h || !bytes) return WAVE2D_ERR_ARG;
    *bytes = (unsigned long long)(h->scheme == 1 ? 4 : 3) * workspace_slice(h);
    return WAVE2D_OK;
}

int wave2d_set_workspace(wave2d_t* h, void* workspace, unsigned long long bytes)
{
    if (!h) return WAVE2D_ERR_ARG;
    if (h->have_initial || h->ran) return WAVE2D_ERR_STATE;   // the ring would lose its contents
    const int nf = h->scheme == 1 ? 4 : 3;
    const size_t slice = workspace_slice(h), fbytes = (size_t)h->pitch * h->n2 * h->elem;
    if (workspace) {
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, workspace) != cudaSuccess ||
            (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)) {
            (void)cudaGetLastError();
            h->err = "wave2d_set_workspace: not device memory";
            return WAVE2D_ERR_ARG;
        }
        if (reinterpret_cast<uintptr_t>(workspace) % 256 != 0 || bytes < (unsigned long long)nf * slice) {
            h->err = "wave2d_set_workspace: needs a 256-byte aligned block of at least wave2d_workspace_bytes() bytes";
            return WAVE2D_ERR_ARG;
        }
    } else if (!h->ext_fields) {
        return WAVE2D_OK;   // already on its own memory
    }
    W2D_CUDA(h, cudaStreamSynchronize(h->stream));
    invalidate_plan(h);   // the TMA descriptors and the graphs name the field addresses
    if (!h->ext_fields)
        for (int b = 0; b < 4; ++b) dev_free(h, h->buf[b], h->buf[b] ? fbytes : 0);
    for (int b = 0; b < 4; ++b) h->buf[b] = nullptr;
    h->ext_fields = false;
    if (workspace) {
        for (int b = 0; b < nf; ++b) h->buf[b] = static_cast<unsigned char*>(workspace) + (size_t)b * slice;
        h->ext_fields = true;
    } else {
        for (int b = 0; b < nf; ++b) {
            int st = dev_alloc(h, &h->buf[b], fbytes);
            if (st) return st;
        }
    }
    for (int b = 0; b < nf; ++b) W2D_CUDA(h, cudaMemsetAsync(h->buf[b], 0, fbytes, h->stream));   // pad columns stay zero
    W2D_CUDA(h, cudaStreamSynchronize(h->stream));
    return WAVE2D_OK;
}

int wave2d_set_initial(wave2d_t* h, const void* phi, const void* psi, long ld)
{
    Range range("wave2d_set_initial");
    if (!h || !phi || ld < h->n1) return WAVE2D_ERR_ARG;
    if (h->scheme == 1) return set_initial_factored(h, phi, psi, ld);
    // w_0 = phi -> buf[1]; psi staged in buf[2]; w_{-1} = phi - (tau/2) psi -> buf[0]   (roles of half-step 0)
    int st = copy_in(h, h->buf[1], phi, ld);
    if (st) return st;
    if (psi) {
        st = copy_in(h, h->buf[2], psi, ld);
        if (st) return st;
    }
    const dim3 blk(128), grd((h->n1 + 127) / 128, h->n2);
    if (h->dtype == WAVE2D_F64)
        wave2d_init_prev<double><<<grd, blk, 0, h->stream>>>((double*)h->buf[0], (const double*)h->buf[1],
                                                             psi ? (const double*)h->buf[2] : nullptr, h->n1, h->n2,
                                                             h->pitch, 0.5 * h->tau);
    else
        wave2d_init_prev<float><<<grd, blk, 0, h->stream>>>((float*)h->buf[0], (const float*)h->buf[1],
                                                            psi ? (const float*)h->buf[2] : nullptr, h->n1, h->n2,
                                                            h->pitch, 0.5 * h->tau);
    W2D_CUDA(h, cudaGetLastError());
    W2D_CUDA(h, cudaMemsetAsync(h->d_k, 0, sizeof(int), h->stream));
    W2D_CUDA(h, cudaMemsetAsync(h->d_tickets, 0, (size_t)2 * SLOTS * sizeof(int), h->stream));   // work queues
    W2D_CUDA(h, cudaStreamSynchronize(h->stream));
    h->have_initial = true;
    h->k = 0;
    h->ran = false;
    return WAVE2D_OK;
}

int wave2d_set_state(wave2d_t* h, int k, const void* u_prev_half, const void* u, long ld)
{
    if (!h || !u_prev_half || !u || ld < h->n1 || k < 0 || k > h->M) return WAVE2D_ERR_ARG;
    if (h->scheme != 0) return WAVE2D_ERR_UNSUPPORTED;   // scheme 1's ring carries (I - ay Dy) u^{k-1}, not a level
    // roles of half-step n = 2k: w_{n-1} = u^{k-1/2} -> buf[n % 3], w_n = u^k -> buf[(n+1) % 3]
    int st = copy_in(h, h->buf[(2 * k) % 3], u_prev_half, ld);
    if (st == WAVE2D_OK) st = copy_in(h, h->buf[(2 * k + 1) % 3], u, ld);
    if (st) return st;
    W2D_CUDA(h, cudaMemsetAsync(h->d_tickets, 0, (size_t)2 * SLOTS * sizeof(int), h->stream));
    W2D_CUDA(h, cudaMemcpyAsync(h->d_k, &k, sizeof(int), cudaMemcpyHostToDevice, h->stream));   // synchronised below
    W2D_CUDA(h, cudaStreamSynchronize(h->stream));
    h->have_initial = true;
    h->k = k;
    return WAVE2D_OK;
}

int wave2d_set_speed(wave2d_t* h, const double* c_half, int count)
{
    if (!h || !c_half || (count != 1 && count != 2 * h->M + 1)) return WAVE2D_ERR_ARG;
    if (h->ran) return WAVE2D_ERR_STATE;
    for (int n = 0; n < count; ++n)
        if (!(c_half[n] > 0.0)) return WAVE2D_ERR_ARG;   // PAPER.md:31, "positive speed function"
    for (int n = 0; n <= 2 * h->M; ++n) h->c_half[n] = count == 1 ? c_half[0] : c_half[n];
    invalidate_plan(h);
    return WAVE2D_OK;
}

int wave2d_set_speed_field(wave2d_t* h, const void* cs, long ld)
{
    if (!h) return WAVE2D_ERR_ARG;
    if (h->ran) return WAVE2D_ERR_STATE;
    if (cs && (ld < h->n1 || h->scheme == 1)) return h->scheme == 1 ? WAVE2D_ERR_UNSUPPORTED : WAVE2D_ERR_ARG;
    if (!cs) {
        invalidate_plan(h);
        h->have_cs = false;
        return WAVE2D_OK;
    }
    // every value must be positive: checked on a host copy BEFORE the handle is touched, so that a
    // rejected field leaves a previously accepted one in place
    const size_t e = h->elem, n1 = h->n1, n2 = h->n2;
    std::vector<unsigned char> host(n1 * n2 * e);
    W2D_CUDA(h, cudaMemcpy2D(host.data(), n1 * e, cs, (size_t)ld * e, n1 * e, n2, cudaMemcpyDefault));
    for (size_t i = 0; i < n1 * n2; ++i) {
        const double v = h->dtype == WAVE2D_F64 ? reinterpret_cast<const double*>(host.data())[i]
                                                : (double)reinterpret_cast<const float*>(host.data())[i];
        if (!(v > 0.0)) return WAVE2D_ERR_ARG;
    }
    const size_t fbytes = (size_t)h->pitch * h->n2 * h->elem;
    if (!h->d_cs) {
        int st = dev_alloc(h, &h->d_cs, fbytes);
        if (st) return st;
    }
    invalidate_plan(h);
    h->have_cs = false;   // until the new field is on the device
    W2D_CUDA(h, cudaMemsetAsync(h->d_cs, 0, fbytes, h->stream));
    W2D_CUDA(h, cudaMemcpy2DAsync(h->d_cs, (size_t)h->pitch * e, host.data(), n1 * e, n1 * e, n2, cudaMemcpyHostToDevice,
                                  h->stream));
    W2D_CUDA(h, cudaStreamSynchronize(h->stream));
    h->have_cs = true;
    return WAVE2D_OK;
}

int wave2d_set_source(wave2d_t* h, const void* s, long ld, const double* g_half, int count)
{
    if (!h) return WAVE2D_ERR_ARG;
    if (h->ran) return WAVE2D_ERR_STATE;
    if (s && (ld < h->n1 || (g_half && count < 2 * h->M))) return WAVE2D_ERR_ARG;
    for (int d = 0; d < 2; ++d) {
        cudaFree(h->src_dev[d]);
        h->src_dev[d] = nullptr;
    }
    h->have_src = false;
    h->g_half.clear();
    invalidate_plan(h);
    if (!s) return WAVE2D_OK;
    // Bring s to the host once, find the window of non-zero values (config 3's sigma = 2h Gaussian underflows to
    // exactly 0 outside ~155^2 points) and keep only that window on the device, in both orientations.
    const size_t e = h->elem, n1 = h->n1, n2 = h->n2;
    std::vector<unsigned char> host(n1 * n2 * e);
    W2D_CUDA(h, cudaMemcpy2D(host.data(), n1 * e, s, (size_t)ld * e, n1 * e, n2, cudaMemcpyDefault));
    auto nz = [&](size_t j, size_t i) {
        return h->dtype == WAVE2D_F64 ? reinterpret_cast<const double*>(host.data())[j * n1 + i] != 0.0
                                      : reinterpret_cast<const float*>(host.data())[j * n1 + i] != 0.0f;
    };
    long i0 = n1, i1 = -1, j0 = n2, j1 = -1;
    for (size_t j = 0; j < n2; ++j)
        for (size_t i = 0; i < n1; ++i)
            if (nz(j, i)) {
                i0 = std::min<long>(i0, i); i1 = std::max<long>(i1, i);
                j0 = std::min<long>(j0, j); j1 = std::max<long>(j1, j);
            }
    if (i1 < 0) return WAVE2D_OK;   // identically zero: no source
    const size_t w = i1 - i0 + 1, hh = j1 - j0 + 1;
    std::vector<unsigned char> nat(w * hh * e), tr(w * hh * e);
    for (size_t j = 0; j < hh; ++j)
        for (size_t i = 0; i < w; ++i) {
            const unsigned char* src = host.data() + ((j0 + j) * n1 + (i0 + i)) * e;
            memcpy(nat.data() + (j * w + i) * e, src, e);
            memcpy(tr.data() + (i * hh + j) * e, src, e);
        }
    int st = dev_alloc(h, &h->src_dev[0], w * hh * e);
    if (st == WAVE2D_OK) st = dev_alloc(h, &h->src_dev[1], w * hh * e);
    if (st) return st;
    W2D_CUDA(h, cudaMemcpy(h->src_dev[0], tr.data(), w * hh * e, cudaMemcpyHostToDevice));
    W2D_CUDA(h, cudaMemcpy(h->src_dev[1], nat.data(), w * hh * e, cudaMemcpyHostToDevice));
    h->win_i0 = (int)i0; h->win_j0 = (int)j0; h->win_w = (int)w; h->win_h = (int)hh;
    h->have_src = true;
    if (g_half) h->g_half.assign(g_half, g_half + 2 * h->M);
    return WAVE2D_OK;
}

int wave2d_run(wave2d_t* h, int steps)
{
    Range range("wave2d_run");
    if (!h || steps < 0) return WAVE2D_ERR_ARG;
    if (!h->have_initial) return WAVE2D_ERR_STATE;
    if ((long long)h->k + steps > h->M) return WAVE2D_ERR_RANGE;
    if (h->scheme == 0 && h->opt_start != 1) return WAVE2D_ERR_UNSUPPORTED;   // (2.9) belongs to the three-level scheme (2.8)
    int st = ensure_plan(h);   // also builds the graphs: wave2d_run(h, 0) prepares everything
    if (st) return st;
    if (steps > 0) h->ran = true;
    if (steps > 0 && h->scheme == 1 && !h->v_ready) {
        st = init_factored_v(h);
        if (st) return st;
    }
    if (h->line_mode) {   // small grid: Algorithm 1's whole loop in one launch of one cluster
        if (steps > 0) {
            st = launch_line_steps(h, steps);
            if (st) return st;
            h->k += steps;
        }
        return WAVE2D_OK;
    }
    // Algorithm 1's loop in chunks of 2^i steps, longest first; each chunk is one graph replay
    // (or, with graph = 0, the same kernel sequence launched directly).
    int left = steps;
    while (left > 0) {
        int i = 0;
        while (i + 1 < NCHUNK && (2 << i) <= left && (2 << i) <= h->opt_graph_steps) ++i;
        const int cs = 1 << i;
        if (h->opt_graph) {
            W2D_CUDA(h, cudaGraphLaunch(h->gexec[i], h->stream));
            h->graph_launches += 1;
        } else {
            st = launch_chunk(h, h->stream, cs);
            if (st) return st;
            h->plain_sweeps += 2 * cs;
        }
        h->launches += kernels_per_chunk(h, cs);
        h->k += cs;
        left -= cs;
    }
    return WAVE2D_OK;
}

int wave2d_get(wave2d_t* h, void* u_out, long ld)
{
    Range range("wave2d_get");
    if (!h) return WAVE2D_ERR_ARG;
    if (h->scheme == 1) return copy_out(h, u_out, ld, h->buf[(h->k - 1) & 3]);   // U^k
    return copy_out(h, u_out, ld, h->buf[(2 * h->k + 1) % 3]);
}

int wave2d_get_prev(wave2d_t* h, void* u_out, long ld)
{
    if (!h) return WAVE2D_ERR_ARG;
    if (h->scheme == 1) {   // the ring carries V^{k-1}, not U^{k-1}; only U^0 is still there before the first solve
        if (h->k == 1 && !h->v_ready) return copy_out(h, u_out, ld, h->buf[3]);
        return WAVE2D_ERR_UNSUPPORTED;
    }
    return copy_out(h, u_out, ld, h->buf[(2 * h->k) % 3]);
}

// Rows [j0, j0 + count) of a time level: 0 = u^k, 1 = u^{k-1/2} (split scheme only).
static int rows_of_level(wave2d_t* h, int level, int j0, int count, void** base)
{
    if (!h || level < 0 || level > 1 || j0 < 0 || count < 1 || j0 + count > h->n2) return WAVE2D_ERR_ARG;
    if (h->scheme != 0) return WAVE2D_ERR_UNSUPPORTED;
    if (!h->have_initial) return WAVE2D_ERR_STATE;
    const int b = level == 0 ? (2 * h->k + 1) % 3 : (2 * h->k) % 3;
    *base = static_cast<unsigned char*>(h->buf[b]) + (size_t)j0 * h->pitch * h->elem;
    return WAVE2D_OK;
}

int wave2d_get_rows(wave2d_t* h, int level, int j0, int count, void* out, long ld)
{
    void* src = nullptr;
    int st = rows_of_level(h, level, j0, count, &src);
    if (st) return st;
    if (!out || ld < h->n1) return WAVE2D_ERR_ARG;
    W2D_CUDA(h, cudaMemcpy2DAsync(out, (size_t)ld * h->elem, src, (size_t)h->pitch * h->elem, (size_t)h->n1 * h->elem, count,
                                  cudaMemcpyDefault, h->stream));
    W2D_CUDA(h, cudaStreamSynchronize(h->stream));
    return WAVE2D_OK;
}

int wave2d_set_rows(wave2d_t* h, int level, int j0, int count, const void* in, long ld)
{
    void* dst = nullptr;
    int st = rows_of_level(h, level, j0, count, &dst);
    if (st) return st;
    if (!in || ld < h->n1) return WAVE2D_ERR_ARG;
    W2D_CUDA(h, cudaMemcpy2DAsync(dst, (size_t)h->pitch * h->elem, in, (size_t)ld * h->elem, (size_t)h->n1 * h->elem, count,
                                  cudaMemcpyDefault, h->stream));
    W2D_CUDA(h, cudaStreamSynchronize(h->stream));   // the caller may reuse `in`
    return WAVE2D_OK;
}

int wave2d_steps_done(const wave2d_t* h, int* k)
{
    if (!h || !k) return WAVE2D_ERR_ARG;
    *k = h->k;
    return WAVE2D_OK;
}

int wave2d_sync(wave2d_t* h)
{
    if (!h) return WAVE2D_ERR_ARG;
    W2D_CUDA(h, cudaStreamSynchronize(h->stream));
    return WAVE2D_OK;
}

int wave2d_get_info(wave2d_t* h, const char* name, double* value)
{
    if (!h || !name || !value) return WAVE2D_ERR_ARG;
    if (!strcmp(name, "pitch")) { *value = (double)h->pitch; return WAVE2D_OK; }
    if (!strcmp(name, "device_bytes")) { *value = (double)h->device_bytes; return WAVE2D_OK; }
    if (!strcmp(name, "launches")) { *value = (double)h->launches; return WAVE2D_OK; }
    if (!strcmp(name, "graph_launches")) { *value = (double)h->graph_launches; return WAVE2D_OK; }
    if (!strcmp(name, "plain_sweeps")) { *value = (double)h->plain_sweeps; return WAVE2D_OK; }
    if (!strcmp(name, "line_launches")) { *value = (double)h->line_launches; return WAVE2D_OK; }
    if (!strcmp(name, "source_window")) { *value = h->have_src ? (double)h->win_w * h->win_h : 0.0; return WAVE2D_OK; }
    int st = ensure_plan(h);
    if (st) return st;
    const size_t len = strlen(name);
    if (len < 3 || name[len - 2] != '_' || (name[len - 1] != 'x' && name[len - 1] != 'y')) return WAVE2D_ERR_ARG;
    const DirPlan& P = h->plan[name[len - 1] == 'y'];
    const std::string key(name, len - 2);
    const bool stream = P.solver == WAVE2D_SOLVER_STREAM;
    if (P.solver == WAVE2D_SOLVER_LINE) {
        if (key == "solver") *value = P.solver;
        else if (key == "rho") *value = P.rho;
        else if (key == "grid") *value = h->line_ctas;
        else if (key == "threads") *value = 32 * LINE_WARPS;
        else if (key == "smem") *value = h->line_smem;
        else if (key == "unit") *value = h->line_unit;
        else if (key == "resident") *value = h->line_resident ? 1 : 0;
        else if (key == "ctas_per_sm") *value = 1;
        else if (key == "chunks") *value = 1;
        else if (key == "halo" || key == "nbk" || key == "kb" || key == "upc" || key == "quota" || key == "static" ||
                 key == "safe") *value = 0;
        else return WAVE2D_ERR_ARG;
        return WAVE2D_OK;
    }
    if (key == "solver") *value = P.solver;
    else if (key == "halo") *value = P.halo;
    else if (key == "rho") *value = P.rho;
    else if (key == "chunks") *value = stream ? (double)P.pieces.size() : 1;
    else if (key == "nbk") *value = stream ? P.nbk : 0;
    else if (key == "kb") *value = stream ? P.kb : 0;
    else if (key == "grid") *value = P.grid;
    else if (key == "ctas_per_sm") *value = stream ? P.ctas_per_sm : 0;
    else if (key == "smem") *value = stream ? P.var->smem : P.ex_smem;
    else if (key == "threads") *value = stream ? P.var->threads : EX_NT;
    else if (key == "unit") *value = stream ? P.var->unit : EX_U;
    else if (key == "strip") *value = stream ? 0 : P.ex_sc;
    else if (key == "upc") *value = stream ? P.quota * P.var->nw : 0;
    else if (key == "quota") *value = stream ? P.quota : 0;
    else if (key == "static") *value = stream ? P.nstatic : 0;
    else if (key == "safe") {
        int c = 0;
        for (const Piece& pc : P.pieces) c += pc.safe != 0;
        *value = c;
    }
    else return WAVE2D_ERR_ARG;
    return WAVE2D_OK;
}

int wave2d_profile_sweeps(wave2d_t* h, int steps, double* ms_x, double* ms_y)
{
    if (!h || steps < 1 || !ms_x || !ms_y) return WAVE2D_ERR_ARG;
    if (!h->have_initial) return WAVE2D_ERR_STATE;
    if ((long long)h->k + steps > h->M) return WAVE2D_ERR_RANGE;
    int st = ensure_plan(h);
    if (st) return st;
    h->ran = true;
    if (h->scheme == 1 && !h->v_ready) {
        st = init_factored_v(h);
        if (st) return st;
    }
    if (h->line_mode) {   // one kernel runs both half-steps of every step: the launch is timed, each sweep gets half
        cudaEvent_t e0, e1;
        W2D_CUDA(h, cudaEventCreate(&e0));
        W2D_CUDA(h, cudaEventCreate(&e1));
        W2D_CUDA(h, cudaEventRecord(e0, h->stream));
        st = launch_line_steps(h, steps);
        if (st) return st;
        W2D_CUDA(h, cudaEventRecord(e1, h->stream));
        W2D_CUDA(h, cudaStreamSynchronize(h->stream));
        float ms = 0.f;
        W2D_CUDA(h, cudaEventElapsedTime(&ms, e0, e1));
        cudaEventDestroy(e0);
        cudaEventDestroy(e1);
        h->k += steps;
        *ms_x = *ms_y = 0.5 * ms / steps;
        return WAVE2D_OK;
    }
    std::vector<cudaEvent_t> ev((size_t)3 * steps);
    for (auto& e : ev) W2D_CUDA(h, cudaEventCreate(&e));
    for (int s = 0; s < steps; ++s) {   // chunks of one step, an event around each sweep
        W2D_CUDA(h, cudaEventRecord(ev[3 * s], h->stream));
        st = launch_half_step(h, h->stream, 0, false);
        if (st) return st;
        W2D_CUDA(h, cudaEventRecord(ev[3 * s + 1], h->stream));
        st = launch_half_step(h, h->stream, 1, h->plan[0].solver == WAVE2D_SOLVER_STREAM);
        if (st) return st;
        W2D_CUDA(h, cudaEventRecord(ev[3 * s + 2], h->stream));
        wave2d_end_chunk<<<1, 2 * SLOTS, 0, h->stream>>>(h->d_k, 1, h->d_tickets);
        W2D_CUDA(h, cudaGetLastError());
        h->launches += kernels_per_chunk(h, 1);
        h->plain_sweeps += 2;
        h->k += 1;
    }
    W2D_CUDA(h, cudaStreamSynchronize(h->stream));
    double sx = 0.0, sy = 0.0;
    for (int s = 0; s < steps; ++s) {
        float a = 0.f, b = 0.f;
        W2D_CUDA(h, cudaEventElapsedTime(&a, ev[3 * s], ev[3 * s + 1]));
        W2D_CUDA(h, cudaEventElapsedTime(&b, ev[3 * s + 1], ev[3 * s + 2]));
        sx += a;
        sy += b;
    }
    for (auto& e : ev) cudaEventDestroy(e);
    *ms_x = sx / steps;
    *ms_y = sy / steps;
    return WAVE2D_OK;
}

int wave2d_get_trace(wave2d_t* h, int dir, unsigned long long* out, int capacity, int* count)
{
    if (!h || dir < 0 || dir > 1 || !out || !count) return WAVE2D_ERR_ARG;
    if (!h->plan_ok || !h->opt_trace || !h->d_trace[dir]) return WAVE2D_ERR_STATE;
    const int g = h->plan[dir].grid;
    *count = g;
    if (capacity < g) return WAVE2D_ERR_ARG;
    W2D_CUDA(h, cudaStreamSynchronize(h->stream));
    W2D_CUDA(h, cudaMemcpy(out, h->d_trace[dir], (size_t)g * 16 * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
    return WAVE2D_OK;
}

// ---- host-only entry points (no device needed): the planning logic, for inspection and tests ----------------
int wave2d_host_scalars(double gamma, double alpha_plus, double alpha_minus, double q, double* out, int capacity,
                        int* count)
{
    if (!out || !count || !(gamma > 0.0) || !(alpha_plus > 0.0) || !(alpha_minus >= 0.0)) return WAVE2D_ERR_ARG;
    *count = ROW_DOUBLES;
    if (capacity < ROW_DOUBLES) return WAVE2D_ERR_ARG;
    fill_row(out, gamma, alpha_plus, alpha_minus, q);
    return WAVE2D_OK;
}

int wave2d_host_decay(int N, double extent, double tau, double c, double gamma, double sigma, double* rho)
{
    if (N < 2 || !(extent > 0.0) || !(tau > 0.0) || !(c > 0.0) || !(gamma > 0.0) || !(sigma > 0.0 && sigma <= 1.0) || !rho)
        return WAVE2D_ERR_ARG;
    const double hd = extent / N;
    double row[ROW_DOUBLES];
    fill_row(row, gamma, sigma * tau * tau * c / (hd * hd), 0.0, 0.0);   // alpha+ as in build_table; alpha-, q do not enter rho
    *rho = row[ROW_RHO];
    return WAVE2D_OK;
}

int wave2d_host_plan(int n, int nlines, int unit, int units_per_stage, int units_per_tile, int nbk, int slots,
                     int fixed_stages, double static_frac, int* pieces, int capacity, int* npieces, int* nstatic,
                     int* cta_off)
{
    if (n < 1 || nlines < 1 || unit < 1 || units_per_stage < 1 || units_per_tile < 1 || nbk < 1 ||
        nbk > units_per_stage || slots < 1 || fixed_stages < 0 || !(static_frac >= 0.0 && static_frac <= 1.0) ||
        !pieces || !npieces || !nstatic || !cta_off)
        return WAVE2D_ERR_ARG;
    DirPlan P;
    P.n = n; P.nlines = nlines; P.nbk = nbk;
    P.npanels = (nlines + 31) / 32;
    P.total_units = (n + unit - 1) / unit;
    const int tail_min = std::min(6, std::max(2, 16384 / (units_per_stage * unit * 32)));   // as plan_dir
    build_pieces(P, units_per_stage, units_per_tile, slots, fixed_stages, static_frac, tail_min, 2.0);
    *npieces = (int)P.pieces.size();
    *nstatic = P.nstatic;
    if (capacity < *npieces) return WAVE2D_ERR_ARG;
    for (size_t i = 0; i < P.pieces.size(); ++i) {
        pieces[4 * i] = P.pieces[i].panel; pieces[4 * i + 1] = P.pieces[i].ua;
        pieces[4 * i + 2] = P.pieces[i].ub; pieces[4 * i + 3] = P.pieces[i].nst;
    }
    for (int c = 0; c <= slots; ++c) cta_off[c] = P.cta_off[c];
    return WAVE2D_OK;
}

const char* wave2d_strerror(int status)
{
    switch (status) {
        case WAVE2D_OK: return "ok";
        case WAVE2D_ERR_ARG: return "invalid argument";
        case WAVE2D_ERR_STATE: return "call not allowed in this state";
        case WAVE2D_ERR_ALLOC: return "allocation failed";
        case WAVE2D_ERR_CUDA: return "CUDA error";
        case WAVE2D_ERR_UNSUPPORTED: return "unsupported size or option";
        case WAVE2D_ERR_RANGE: return "more than M steps requested";
        default: return "unknown status";
    }
}

const char* wave2d_last_error(const wave2d_t* h) { return h ? h->err.c_str() : ""; }

}  // extern "C"

// =====================================================================================================
// wave2d_small_steps_static (include/wave2d.h): the small-grid step loop for callers that must not allocate.
//
// The handle path above cudaMallocs its working memory (wave2d_create: three time levels and the counters; the first
// run: the scalar table).  Some users of a small-grid solver cannot afford that: a plug-in inside a framework whose
// caching allocator has already reserved the GPU's memory (a raw cudaMalloc then fails although the framework shows
// free space), a service with a device-memory budget fixed at start-up, a control loop that other streams share the
// GPU with (cudaMalloc / cudaFree synchronise the whole device and stall them).  For these the working memory of ONE
// kernel -- the small-grid kernel of line.cuh, whose scratch is the ring of three time levels plus the two scalar rows
// -- is the file-scope array below: it is part of the library image, so every GPU that loads libwave2d.so holds its
// 1.5 MiB from module load until the process exits, and no call ever allocates or frees anything.
//
// The price: ONE array per device, shared by every call in the process.  It keeps whatever the last call left in it
// (each call rewrites everything it later reads, see the kernel's prologue), and two calls whose kernels overlap on the
// GPU (different streams without an event between them, or two host threads) overwrite each other's time levels.
// =====================================================================================================
#include <cstdarg>
#include <mutex>

namespace w2d_static {
constexpr int NMAX = 32 * 8;                                                   // unknowns per line, either direction
constexpr size_t FIELD_BYTES = (size_t)NMAX * NMAX * sizeof(double);           // one time level at the largest size
constexpr size_t TABLE_BYTES = (size_t)2 * w2d::ROW_DOUBLES * sizeof(double);  // scalar rows of the x and y half-step
constexpr size_t SCRATCH_BYTES = 3 * FIELD_BYTES + TABLE_BYTES;                // 1 581 184 bytes
static_assert(NMAX <= w2d::KMAX, "every pivot of a line is tabulated");
}  // namespace w2d_static

// In HOST code this name is only a handle for cudaGetSymbolAddress: its host-side address is not device memory, and a
// kernel handed `wave2d_static_scratch` directly would fault (or, where the GPU can reach host memory, quietly work on
// the wrong bytes).  static_device() below asks the runtime for the device address, per device.
static __device__ __align__(256) unsigned char wave2d_static_scratch[w2d_static::SCRATCH_BYTES];

namespace {

struct StaticArgs {
    unsigned char* scratch;   // DEVICE address of wave2d_static_scratch on the device that runs the kernel
    const void* in_prev;      // caller: u^{k-1/2}      } n2 rows of n1 values, row stride ld (elements)
    const void* in_cur;       // caller: u^k            }
    void* out_cur;            // caller: u^{k+nsteps}
    void* out_prev;           // caller: u^{k+nsteps-1/2}, or NULL
    long long ld, pitch;      // elements; pitch = row stride inside the scratch, a multiple of 16
    int n1, n2, nsteps;
    double g2;                // 2 gamma
    double rows[2][ROW_DOUBLES];   // [0]: x half-steps, [1]: y half-steps (constant speed: two rows serve every step)
};

// wave2d_line_steps (line.cuh) with its global working memory inside `a.scratch` instead of cudaMalloc'd buffers:
//   scratch + b * FIELD_BYTES, b = 0..2   the ring of time levels, roles by roles_of(nh, 3), rows a.pitch apart
//   scratch + 3 * FIELD_BYTES             the two scalar rows (copied from the kernel parameters by CTA 0)
// Prologue: the caller's two levels are copied into ring buffers 0 and 1 with the pad columns [n1, pitch) written as
// zeros -- the only part of the scratch that must start at zero (a row's right-hand ghost value, (2.10)); ring buffer 2
// is written by the first x half-step over the full pitch before anything reads it, so nothing a previous call left
// behind is ever read.  Epilogue: the last two levels go to the caller's arrays.  Constant speed, no source, split
// scheme (2.11)-(2.12) with gamma = 2, kappa = 1/2; the line solve is solve_line_warp, as in the handle path.
// grid = one cluster; block = 32 * W threads; dynamic shared memory: two strips [16][32 U + 1] of T.
template <typename T, int U, int W>
__global__ void __launch_bounds__(32 * W, 1) wave2d_line_steps_static(const __grid_constant__ StaticArgs a)
{
    constexpr int V = 16 / (int)sizeof(T), NV = U / V, SC = 16, KC = SC / V, RP = 32 * U + 1;
    extern __shared__ __align__(16) unsigned char static_smem[];
    T* const s_prev = reinterpret_cast<T*>(static_smem);
    T* const s_cur = s_prev + SC * RP;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int cta = (int)cluster_ctarank(), ncta = (int)cluster_nctarank();
    const int p0 = U * lane;
    const T g2 = static_cast<T>(a.g2);
    auto level = [&](int b) { return reinterpret_cast<T*>(a.scratch + (size_t)b * w2d_static::FIELD_BYTES); };
    double* const tab = reinterpret_cast<double*>(a.scratch + 3 * w2d_static::FIELD_BYTES);

    // ---- prologue: scalar rows and the caller's two time levels into the scratch
    if (cta == 0)
        for (int i = threadIdx.x; i < 2 * ROW_DOUBLES; i += 32 * W) tab[i] = a.rows[i / ROW_DOUBLES][i % ROW_DOUBLES];
    {
        const T* const ip = static_cast<const T*>(a.in_prev);
        const T* const ic = static_cast<const T*>(a.in_cur);
        T* const b0 = level(0);   // roles_of(0, 3): w_{-1} = ring 0, w_0 = ring 1
        T* const b1 = level(1);
        for (int j = cta * W + warp; j < a.n2; j += ncta * W)
            for (int i = lane; i < a.pitch; i += 32) {
                const bool in = i < a.n1;
                b0[j * a.pitch + i] = in ? ip[j * a.ld + i] : T(0);
                b1[j * a.pitch + i] = in ? ic[j * a.ld + i] : T(0);
            }
    }
    cluster_barrier();

    for (int nh = 0; nh < 2 * a.nsteps; ++nh) {
        const int d = nh & 1;
        const double* row = tab + d * ROW_DOUBLES;
        const Roles R = roles_of(nh, 3);
        const T* const prev = level(R.prev);
        const T* const cur = level(R.cur);
        T* const out = level(R.out);
        const int n = d == 0 ? a.n1 : a.n2, nlines = d == 0 ? a.n2 : a.n1;
        const T am = static_cast<T>(a.rows[d][ROW_AM]), c1 = static_cast<T>(a.rows[d][ROW_C1]);
        T cp[U], iv[U], qs[U];
#pragma unroll
        for (int e = 0; e < U; ++e) {            // beyond the line: cp = inv = 0 decouples the padding (x = 0 there)
            const bool in = p0 + e < n;
            cp[e] = in ? static_cast<T>(__ldcg(row + ROW_CP + p0 + e)) : T(0);
            iv[e] = in ? static_cast<T>(__ldcg(row + ROW_INVP + p0 + e)) : T(0);
            qs[e] = T(0);                        // no source
        }
        if (d == 0) {
            // ---- x half-step: one warp per grid row, lanes along the row
            const bool inrow = p0 < a.pitch;
            for (int j = cta * W + warp; j < nlines; j += ncta * W) {
                T wp[U], wc[U];
#pragma unroll
                for (int e = 0; e < U; ++e) wp[e] = wc[e] = T(0);
                const long long o = static_cast<long long>(j) * a.pitch + p0;
                if (inrow) {
#pragma unroll
                    for (int c = 0; c < NV; ++c) {
                        ldcg16(prev + o + c * V, wp + c * V);
                        ldcg16(cur + o + c * V, wc + c * V);
                    }
                }
                solve_line_warp<T, U>(wp, wc, qs, cp, iv, am, c1, g2, false, lane);
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
                    const long long o = static_cast<long long>(r) * a.pitch + c0 + kc * V;   // c0 + 16 <= pitch
                    ldcg16(prev + o, vp);
                    ldcg16(cur + o, vc);
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        s_prev[(kc * V + e) * RP + r] = vp[e];
                        s_cur[(kc * V + e) * RP + r] = vc[e];
                    }
                }
                __syncthreads();
                for (int w = warp; w < SC; w += W) {            // warp = grid column c0 + w (pad columns solve zeros)
                    T wp[U], wc[U];
#pragma unroll
                    for (int e = 0; e < U; ++e) {
                        const bool in = p0 + e < n;
                        wp[e] = in ? s_prev[w * RP + p0 + e] : T(0);
                        wc[e] = in ? s_cur[w * RP + p0 + e] : T(0);
                    }
                    solve_line_warp<T, U>(wp, wc, qs, cp, iv, am, c1, g2, false, lane);
#pragma unroll
                    for (int e = 0; e < U; ++e)
                        if (p0 + e < n) s_cur[w * RP + p0 + e] = wc[e];
                }
                __syncthreads();
                for (int r = r0; r < n; r += (32 * W) / KC) {
                    T vo[V];
#pragma unroll
                    for (int e = 0; e < V; ++e) vo[e] = s_cur[(kc * V + e) * RP + r];
                    st16(out + static_cast<long long>(r) * a.pitch + c0 + kc * V, vo);
                }
                __syncthreads();
            }
        }
        cluster_barrier();   // the half-step's stores are visible to every CTA of the cluster
    }

    // ---- epilogue: roles_of(2 nsteps, 3): "cur" = u^{k+nsteps}, "prev" = u^{k+nsteps-1/2}
    {
        const Roles R = roles_of(2 * a.nsteps, 3);
        const T* const fc = level(R.cur);
        const T* const fp = level(R.prev);
        T* const oc = static_cast<T*>(a.out_cur);
        T* const op = static_cast<T*>(a.out_prev);
        for (int j = cta * W + warp; j < a.n2; j += ncta * W)
            for (int i = lane; i < a.n1; i += 32) {
                oc[j * a.ld + i] = __ldcg(fc + j * a.pitch + i);
                if (op != nullptr) op[j * a.ld + i] = __ldcg(fp + j * a.pitch + i);
            }
    }
}

template <typename T, int U>
const void* static_kernel() { return reinterpret_cast<const void*>(&wave2d_line_steps_static<T, U, LINE_WARPS>); }

const void* static_kernel_of(int dtype, int U)
{
    if (dtype == WAVE2D_F64) return U == 4 ? static_kernel<double, 4>() : static_kernel<double, 8>();
    return U == 4 ? static_kernel<float, 4>() : static_kernel<float, 8>();
}

int static_smem_bytes(int dtype, int U) { return 2 * 16 * (32 * U + 1) * (dtype == WAVE2D_F64 ? 8 : 4); }

// Per-device set-up, done by the first call on a device with that device current: the DEVICE address of the scratch
// array (every device has its own copy of a __device__ variable, so the address is asked for per device) and the
// opt-in to more than 48 KB of dynamic shared memory for the four instantiations.  Fixed-size table, no heap.
constexpr int STATIC_MAX_DEVICES = 64;
struct StaticDevice {
    bool ready = false;
    unsigned char* scratch = nullptr;
};
StaticDevice g_static_device[STATIC_MAX_DEVICES];
std::mutex g_static_mutex;

void static_msg(char* errbuf, int errbuf_len, const char* fmt, ...)
{
    if (!errbuf || errbuf_len <= 0) return;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(errbuf, (size_t)errbuf_len, fmt, ap);
    va_end(ap);
}

int static_device(int dev, unsigned char** scratch, char* errbuf, int errbuf_len)
{
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) {
        static_msg(errbuf, errbuf_len, "device ordinal %d: the static path serves devices 0..%d", dev, STATIC_MAX_DEVICES - 1);
        return WAVE2D_ERR_UNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice& D = g_static_device[dev];
    if (!D.ready) {
        int major = 0;
        cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e == cudaSuccess && major != 10) {
            static_msg(errbuf, errbuf_len, "device %d is not an sm_100 device: there is no other code path", dev);
            return WAVE2D_ERR_CUDA;
        }
        unsigned char* ptr = nullptr;
        if (e == cudaSuccess) e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), wave2d_static_scratch);
        for (int dt = 0; dt < 2 && e == cudaSuccess; ++dt)
            for (int U = 4; U <= 8 && e == cudaSuccess; U += 4)
                e = cudaFuncSetAttribute(static_kernel_of(dt, U), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_smem_bytes(dt, U));
        if (e != cudaSuccess || ptr == nullptr) {
            static_msg(errbuf, errbuf_len, "set-up on device %d: %s", dev, cudaGetErrorString(e));
            (void)cudaGetLastError();
            return WAVE2D_ERR_CUDA;
        }
        D.scratch = ptr;
        D.ready = true;
    }
    *scratch = D.scratch;
    return WAVE2D_OK;
}

// a pointer the kernel can dereference on device `dev`?  (cudaPointerGetAttributes allocates nothing)
bool static_on_device(const void* p, int dev)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    return at.type == cudaMemoryTypeManaged || (at.type == cudaMemoryTypeDevice && at.device == dev);
}

}  // namespace

extern "C" int wave2d_small_steps_static(int N1, int N2, double l, double tau, double c, int steps, int dtype,
                                         const void* u_prev_half, const void* u, void* u_out, void* u_prev_out, long ld,
                                         void* cuda_stream, char* errbuf, int errbuf_len)
{
    if (errbuf && errbuf_len > 0) errbuf[0] = '\0';
    if (N1 < 2 || N2 < 2 || !(l > 0.0) || !(tau > 0.0) || !(c > 0.0) || steps < 1 ||
        (dtype != WAVE2D_F64 && dtype != WAVE2D_F32) || !u_prev_half || !u || !u_out || ld < N1 - 1) {
        static_msg(errbuf, errbuf_len, "wave2d_small_steps_static: need N1, N2 >= 2, l, tau, c > 0, steps >= 1, a valid dtype, "
                   "non-NULL u_prev_half, u, u_out and ld >= N1 - 1");
        return WAVE2D_ERR_ARG;
    }
    const int n1 = N1 - 1, n2 = N2 - 1;
    if (n1 > w2d_static::NMAX || n2 > w2d_static::NMAX) {
        static_msg(errbuf, errbuf_len, "wave2d_small_steps_static: %d x %d unknowns, but the static scratch holds lines of at most "
                   "%d unknowns in each direction (N1, N2 <= %d); larger grids need a wave2d_create handle", n1, n2,
                   w2d_static::NMAX, w2d_static::NMAX + 1);
        return WAVE2D_ERR_UNSUPPORTED;
    }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        static_msg(errbuf, errbuf_len, "wave2d_small_steps_static: no CUDA device (there is no CPU fallback)");
        (void)cudaGetLastError();
        return WAVE2D_ERR_CUDA;
    }
    unsigned char* scratch = nullptr;
    int st = static_device(dev, &scratch, errbuf, errbuf_len);
    if (st) return st;
    if (!static_on_device(u_prev_half, dev) || !static_on_device(u, dev) || !static_on_device(u_out, dev) ||
        (u_prev_out && !static_on_device(u_prev_out, dev))) {
        static_msg(errbuf, errbuf_len, "wave2d_small_steps_static: every field must be DEVICE memory of the current device %d "
                   "(a host array would need a staging buffer, which this call may not allocate)", dev);
        return WAVE2D_ERR_ARG;
    }

    StaticArgs a;   // 8.4 KB of kernel parameters, on the stack
    a.scratch = scratch;
    a.in_prev = u_prev_half; a.in_cur = u; a.out_cur = u_out; a.out_prev = u_prev_out;
    a.ld = ld;
    a.pitch = (n1 + 15) / 16 * 16;
    a.n1 = n1; a.n2 = n2; a.nsteps = steps;
    const double gamma = 2.0, sigma = 0.5, t2 = tau * tau;
    a.g2 = 2.0 * gamma;
    for (int d = 0; d < 2; ++d) {   // as build_table for scheme 0 with a constant speed and no source
        const double hd = d == 0 ? l / N1 : l / N2;
        fill_row(a.rows[d], gamma, sigma * t2 * c / (hd * hd), (1.0 - sigma) * t2 * c / (hd * hd), 0.0);
    }
    const int nmax = std::max(n1, n2);
    const int U = nmax <= 32 * 4 ? 4 : 8;
    const int ctas = std::max(1, std::min(8, std::max((n2 + LINE_WARPS - 1) / LINE_WARPS, (n1 + 15) / 16)));
    void* args[1] = {&a};
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(ctas);
    cfg.blockDim = dim3(32 * LINE_WARPS);
    cfg.dynamicSmemBytes = static_smem_bytes(dtype, U);
    cfg.stream = static_cast<cudaStream_t>(cuda_stream);
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = ctas;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    const cudaError_t e = cudaLaunchKernelExC(&cfg, static_kernel_of(dtype, U), args);
    if (e != cudaSuccess) {
        static_msg(errbuf, errbuf_len, "wave2d_small_steps_static: launch: %s", cudaGetErrorString(e));
        (void)cudaGetLastError();
        return WAVE2D_ERR_CUDA;
    }
    return WAVE2D_OK;
}
