/*
 * wave2d_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU implementation (fp64, Thomas algorithm, OpenMP over lines)
 * of the ADI / locally-one-dimensional time stepping of
 *
 *     u_tt - c(t) (u_xx + u_yy) = f(t,x,y)   on [0,l]^2,  u = 0 on the boundary     ((2.1)-(2.5))
 *
 * as split in PAPER.md:79-85, eqs (2.11) (implicit in x) and (2.12) (implicit in y), and driven by
 * the loop of Algorithm 1.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference leg may call this file.  It shares no code, header, table or
 * constant with the CUDA path under paper_2006_10142_b200/ and uses a different algorithm
 * (Thomas elimination per line with explicit a,b,c,f arrays; the GPU solves unit-local scalar-pivot
 * recurrences joined by carry series).
 *
 * Notation:
 *   n1 = N1-1, n2 = N2-1      unknowns per x-line / y-line; h_d = l/N_d
 *   w_n                       grid function at half-level n (t = n*tau/2);
 *                             w_{2k} = u^k, w_{2k+1} = u^{k+1/2}, w_{-1} = u^{-1/2}
 *   half-step n -> n+1        implicit in x if n is even, in y if n is odd
 *   storage                   interior points only, [j][i] with i (x) fastest, zero ghosts (2.10)
 *
 * One half-step, multiplied through by tau^2 (reading A2 of DESIGN.md: gamma = 2, kappa = 1/2 is
 * the consistent LOD form; gamma = 1, kappa = 1 is the scheme exactly as printed):
 *
 *   gamma (x_p - 2 w_n[p] + w_{n-1}[p])
 *      - ap (x_{p+1} - 2 x_p + x_{p-1}) - am (w_{n-1}[p+1] - 2 w_{n-1}[p] + w_{n-1}[p-1])
 *      = kappa tau^2 g_n s[p]
 *
 *   ap = tau^2 c_{n+1} / (2 h_d^2),   am = tau^2 c_{n-1} / (2 h_d^2),   c_{-1} := c_0.
 *
 * i.e. the tridiagonal system   a_p x_{p-1} + b_p x_p + c_p x_{p+1} = f_p   with
 *   a_p = c_p = -ap,  b_p = gamma + 2 ap,
 *   f_p = gamma (2 w_n[p] - w_{n-1}[p]) + am (w_{n-1}[p-1] - 2 w_{n-1}[p] + w_{n-1}[p+1]) + kappa tau^2 g_n s[p].
 *
 * A second scheme (option "scheme" = 1, oracle_factored_step below) is the factorised form of the unsplit
 * scheme (2.8); it has its own pins (tests/test_oracle_factored.py).
 *
 * A variable speed c(t) cs(x,y) (oracle_half_step_var) has its pins in
 * tests/test_oracle_varspeed.py.
 *
 * Two more options of SURVEY.md 8f NEXT-4 (pins in tests/test_oracle_variants.py):
 *   "sigma"  weight of the implicit operator in the split scheme: ap = sigma tau^2 c_{n+1} / h_d^2,
 *            am = (1 - sigma) tau^2 c_{n-1} / h_d^2.  sigma = 1/2 is (2.11)-(2.12); sigma = 1 (with gamma = 1, c = 1) is
 *            the system Listing 1 prints: a = c = tau^2, b = 2 tau^2 + h^2, f = h^2 u^{k-1} - 2 h^2 u^k.
 *   "start"  2: second-order start of the three-level scheme (2.8) (scheme 1) for psi != 0 or f != 0:
 *            u^1 = phi + tau psi + (tau^2 / 2) (c^0 Lap_h phi + f^0), the Taylor value with u_tt from (2.1);
 *            1 (default): (2.9) as printed, u^1 = phi + tau psi.
 *
 * Parity pins (tests/test_oracle_*.py): dense LU of the Kronecker system on tiny grids, the exact
 * discrete modal recurrence, the PDE standing wave (observed order 1), forced response, tridiagonal
 * residuals, linearity / reflection invariants.  Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_ERR_ARG (-1)
#define ORACLE_ERR_STATE (-2)
#define ORACLE_ERR_ALLOC (-3)
#define ORACLE_ERR_RANGE (-6)

/* ------------------------------------------------------------------------------------------------
 * Thomas algorithm (no pivoting) for  a[p] x[p-1] + b[p] x[p] + c[p] x[p+1] = f[p],  p = 0..n-1,
 * with x[-1] = x[n] = 0 (a[0] and c[n-1] are never read).  cp, fp: caller-provided scratch of n.
 * This is "call function CR(a_i, b_i, c_i, f_i, y_i, n)" of Algorithm 1 with the
 * line solver replaced by plain Gaussian elimination of the same system.
 * ---------------------------------------------------------------------------------------------- */
void oracle_thomas(int n, const double *a, const double *b, const double *c, const double *f,
                   double *x, double *cp, double *fp)
{
    if (n <= 0) return;
    cp[0] = c[0] / b[0];
    fp[0] = f[0] / b[0];
    for (int p = 1; p < n; ++p) {
        double den = b[p] - a[p] * cp[p - 1];
        cp[p] = c[p] / den;
        fp[p] = (f[p] - a[p] * fp[p - 1]) / den;
    }
    x[n - 1] = fp[n - 1];
    for (int p = n - 2; p >= 0; --p) x[p] = fp[p] - cp[p] * x[p + 1];
}

/* ------------------------------------------------------------------------------------------------
 * One half-step  w_{n-1}, w_n -> w_{n+1}   (eq (2.11) if dir == 0, eq (2.12) if dir == 1).
 *   dir   0: lines along x (one per grid row j),   1: lines along y (one per grid column i)
 *   ap,am the two operator weights defined above (already divided by 2 h_d^2 and times tau^2)
 *   q     kappa * tau^2 * g_n  (source weight); s may be NULL (no source)
 * Arrays are n2 rows x n1 columns, contiguous (ld = n1).
 * ---------------------------------------------------------------------------------------------- */
void oracle_half_step(int n1, int n2, int dir, double ap, double am, double gamma, double q,
                      const double *w_prev, const double *w_cur, const double *s, double *w_next)
{
    const int nlines = dir == 0 ? n2 : n1;   /* number of independent systems            */
    const int n = dir == 0 ? n1 : n2;        /* unknowns per system                      */
    const long step = dir == 0 ? 1 : n1;     /* memory stride between neighbours on line */
    const long lstep = dir == 0 ? n1 : 1;    /* memory stride between lines              */

#pragma omp parallel
    {
        double *a = (double *)malloc(sizeof(double) * 7 * (size_t)(n > 0 ? n : 1));
        double *b = a + n, *c = b + n, *f = c + n, *x = f + n, *cp = x + n, *fp = cp + n;
#pragma omp for schedule(static)
        for (int line = 0; line < nlines; ++line) {
            const double *wp = w_prev + line * lstep;
            const double *wc = w_cur + line * lstep;
            const double *sp = s ? s + line * lstep : NULL;
            /* "calculate tridiagonal system elements a_i, b_i, c_i, f_i" */
            for (int p = 0; p < n; ++p) {
                double wm = p > 0 ? wp[(p - 1) * step] : 0.0;     /* zero Dirichlet ghost, (2.10) */
                double wq = p < n - 1 ? wp[(p + 1) * step] : 0.0;
                double w0 = wp[p * step];
                a[p] = -ap;
                b[p] = gamma + 2.0 * ap;
                c[p] = -ap;
                f[p] = gamma * (2.0 * wc[p * step] - w0) + am * (wm - 2.0 * w0 + wq);
                if (sp) f[p] += q * sp[p * step];
            }
            oracle_thomas(n, a, b, c, f, x, cp, fp);
            double *wn = w_next + line * lstep;
            for (int p = 0; p < n; ++p) wn[p * step] = x[p];
        }
        free(a);
    }
}

/* ------------------------------------------------------------------------------------------------
 * Variable speed (reading R16).  Algorithm 1 computes the tridiagonal elements
 * a_i, b_i, c_i, f_i point by point; with a speed c(t) cs(x,y) -- separable like the source
 * f = g(t) s(x,y) of PAPER.md:33 -- the weights of (2.11)/(2.12) are taken at the point p of the equation:
 *
 *   gamma (x_p - 2 w_n[p] + w_{n-1}[p])
 *      - ap cs[p] (x_{p+1} - 2 x_p + x_{p-1}) - am cs[p] (w_{n-1}[p+1] - 2 w_{n-1}[p] + w_{n-1}[p-1])
 *      = kappa tau^2 g_n s[p]
 *
 * i.e.  a_p = c_p = -ap cs[p],  b_p = gamma + 2 ap cs[p]  (a non-Toeplitz, non-symmetric, strictly diagonally
 * dominant system per line).  ap, am, q as in oracle_half_step; cs: n2 x n1, every value > 0.
 * ---------------------------------------------------------------------------------------------- */
void oracle_half_step_var(int n1, int n2, int dir, double ap, double am, double gamma, double q, const double *cs,
                          const double *w_prev, const double *w_cur, const double *s, double *w_next)
{
    const int nlines = dir == 0 ? n2 : n1;
    const int n = dir == 0 ? n1 : n2;
    const long step = dir == 0 ? 1 : n1;
    const long lstep = dir == 0 ? n1 : 1;

#pragma omp parallel
    {
        double *a = (double *)malloc(sizeof(double) * 7 * (size_t)(n > 0 ? n : 1));
        double *b = a + n, *c = b + n, *f = c + n, *x = f + n, *cp = x + n, *fp = cp + n;
#pragma omp for schedule(static)
        for (int line = 0; line < nlines; ++line) {
            const double *wp = w_prev + line * lstep;
            const double *wc = w_cur + line * lstep;
            const double *cl = cs + line * lstep;
            const double *sp = s ? s + line * lstep : NULL;
            for (int p = 0; p < n; ++p) {
                double wm = p > 0 ? wp[(p - 1) * step] : 0.0;     /* zero Dirichlet ghost, (2.10) */
                double wq = p < n - 1 ? wp[(p + 1) * step] : 0.0;
                double w0 = wp[p * step];
                double app = ap * cl[p * step], amp = am * cl[p * step];
                a[p] = -app;
                b[p] = gamma + 2.0 * app;
                c[p] = -app;
                f[p] = gamma * (2.0 * wc[p * step] - w0) + amp * (wm - 2.0 * w0 + wq);
                if (sp) f[p] += q * sp[p * step];
            }
            oracle_thomas(n, a, b, c, f, x, cp, fp);
            double *wn = w_next + line * lstep;
            for (int p = 0; p < n; ++p) wn[p * step] = x[p];
        }
        free(a);
    }
}

/* ------------------------------------------------------------------------------------------------
 * Scheme 1: the factorised form of the UNSPLIT three-level scheme (2.8).
 * (2.8) times tau^2 reads, with a_d^+- = tau^2 c^{k+-1} / (2 h_d^2) and D_d the undivided second difference
 * along d with zero Dirichlet ghosts (2.10),
 *
 *     (I - ax+ Dx - ay+ Dy) u^{k+1} = 2 u^k - (I - ax- Dx - ay- Dy) u^{k-1} + tau^2 f^k.
 *
 * Replacing both operators by their products (the alternating-direction factorisation; the added terms
 * a^2 Dx Dy u are O(tau^4)) gives one x solve and one y solve per step:
 *
 *     z = (I - ay- Dy) u^{k-1}                                   explicit
 *     R = 2 u^k - (I - ax- Dx) z + tau^2 g_k s                   explicit
 *     (I - ax+ Dx) v = R                                         Thomas on every grid row
 *     (I - ay+ Dy) u^{k+1} = v                                   Thomas on every grid column
 *
 * Every operator is applied / inverted literally here, point by point.  Arrays: n2 rows x n1 columns.
 * ---------------------------------------------------------------------------------------------- */
void oracle_factored_step(int n1, int n2, double axp, double axm, double ayp, double aym, double q,
                          const double *u_prev, const double *u_cur, const double *s, double *u_next)
{
    const size_t npts = (size_t)n1 * (size_t)n2;
    double *z = (double *)malloc(sizeof(double) * 2 * (npts ? npts : 1));
    double *v = z + npts;
#pragma omp parallel for schedule(static)
    for (int j = 0; j < n2; ++j)
        for (int i = 0; i < n1; ++i) {
            const double up = j > 0 ? u_prev[(size_t)(j - 1) * n1 + i] : 0.0;
            const double dn = j < n2 - 1 ? u_prev[(size_t)(j + 1) * n1 + i] : 0.0;
            const double c0 = u_prev[(size_t)j * n1 + i];
            z[(size_t)j * n1 + i] = c0 - aym * (up - 2.0 * c0 + dn);
        }
#pragma omp parallel
    {
        const int nmax = n1 > n2 ? n1 : n2;
        double *a = (double *)malloc(sizeof(double) * 7 * (size_t)(nmax > 0 ? nmax : 1));
        double *b = a + nmax, *c = b + nmax, *f = c + nmax, *x = f + nmax, *cp = x + nmax, *fp = cp + nmax;
#pragma omp for schedule(static)
        for (int j = 0; j < n2; ++j) {   /* x solve, one system per grid row */
            const double *zr = z + (size_t)j * n1;
            for (int i = 0; i < n1; ++i) {
                const double zl = i > 0 ? zr[i - 1] : 0.0, zq = i < n1 - 1 ? zr[i + 1] : 0.0;
                a[i] = -axp; b[i] = 1.0 + 2.0 * axp; c[i] = -axp;
                f[i] = 2.0 * u_cur[(size_t)j * n1 + i] - (zr[i] - axm * (zl - 2.0 * zr[i] + zq));
                if (s) f[i] += q * s[(size_t)j * n1 + i];
            }
            oracle_thomas(n1, a, b, c, f, x, cp, fp);
            memcpy(v + (size_t)j * n1, x, sizeof(double) * (size_t)n1);
        }
#pragma omp for schedule(static)
        for (int i = 0; i < n1; ++i) {   /* y solve, one system per grid column */
            for (int j = 0; j < n2; ++j) {
                a[j] = -ayp; b[j] = 1.0 + 2.0 * ayp; c[j] = -ayp;
                f[j] = v[(size_t)j * n1 + i];
            }
            oracle_thomas(n2, a, b, c, f, x, cp, fp);
            for (int j = 0; j < n2; ++j) u_next[(size_t)j * n1 + i] = x[j];
        }
        free(a);
    }
    free(z);
}

/* ------------------------------------------------------------------------------------------------
 * Handle API, mirroring the wave2d_* C ABI (include/wave2d.h) with host pointers and fp64 only.
 * ---------------------------------------------------------------------------------------------- */
typedef struct oracle_wave2d_s {
    int N1, N2, n1, n2, M;
    double l, tau, gamma, kappa;
    double *c_half;   /* 2M+1 samples c(n tau/2)                                   */
    double *g_half;   /* 2M samples g(n tau/2), or NULL meaning g == 1             */
    double *s;        /* n2 x n1 source shape, or NULL (no source)                 */
    double *cs;       /* n2 x n1 spatial speed factor, or NULL (c = c(t) only)     */
    double *w[3];     /* w[0] = w_{n-1}, w[1] = w_n, w[2] = scratch for w_{n+1}     */
    int have_initial; /* set_initial called                                        */
    int n_done;       /* half-steps taken so far (scheme 1: 2 x the time level k)  */
    int scheme;       /* 0: split scheme (2.11)-(2.12); 1: factorised (2.8)        */
    double sigma;     /* weight of the implicit operator in the split scheme (1/2)   */
    int start;        /* scheme 1: 1 = (2.9) as printed, 2 = second-order start      */
    int start_done;   /* the second-order term has been added (at the first run)     */
} oracle_wave2d_t;

int oracle_wave2d_create(oracle_wave2d_t **out, int N1, int N2, double l, double tau, int M)
{
    if (!out || N1 < 2 || N2 < 2 || !(l > 0.0) || !(tau > 0.0) || M < 0) return ORACLE_ERR_ARG;
    oracle_wave2d_t *h = (oracle_wave2d_t *)calloc(1, sizeof(*h));
    if (!h) return ORACLE_ERR_ALLOC;
    h->N1 = N1; h->N2 = N2; h->n1 = N1 - 1; h->n2 = N2 - 1; h->M = M;
    h->l = l; h->tau = tau;
    h->gamma = 2.0;   /* DESIGN.md reading A2: consistent LOD form */
    h->kappa = 0.5;
    h->sigma = 0.5;
    h->start = 1;
    size_t npts = (size_t)h->n1 * (size_t)h->n2;
    h->c_half = (double *)malloc(sizeof(double) * (size_t)(2 * M + 1));
    for (int k = 0; k < 3; ++k) h->w[k] = (double *)calloc(npts, sizeof(double));
    if (!h->c_half || !h->w[0] || !h->w[1] || !h->w[2]) return ORACLE_ERR_ALLOC;
    for (int n = 0; n <= 2 * M; ++n) h->c_half[n] = 1.0;   /* default c == 1 */
    *out = h;
    return ORACLE_OK;
}

void oracle_wave2d_destroy(oracle_wave2d_t *h)
{
    if (!h) return;
    free(h->c_half); free(h->g_half); free(h->s); free(h->cs);
    for (int k = 0; k < 3; ++k) free(h->w[k]);
    free(h);
}

/* gamma / kappa of reading A2.  name: "gamma" or "kappa". */
int oracle_wave2d_set_option(oracle_wave2d_t *h, const char *name, double value)
{
    if (!h || !name) return ORACLE_ERR_ARG;
    if (h->n_done > 0) return ORACLE_ERR_STATE;
    if (!strcmp(name, "gamma")) { if (!(value > 0.0)) return ORACLE_ERR_ARG; h->gamma = value; return ORACLE_OK; }
    if (!strcmp(name, "kappa")) { h->kappa = value; return ORACLE_OK; }
    if (!strcmp(name, "sigma")) { if (!(value > 0.0 && value <= 1.0)) return ORACLE_ERR_ARG; h->sigma = value; return ORACLE_OK; }
    if (!strcmp(name, "start")) { if (value != 1.0 && value != 2.0) return ORACLE_ERR_ARG; h->start = (int)value; return ORACLE_OK; }
    if (!strcmp(name, "scheme")) {   /* before set_initial */
        if ((value != 0.0 && value != 1.0) || h->have_initial) return ORACLE_ERR_ARG;
        h->scheme = (int)value;
        return ORACLE_OK;
    }
    return ORACLE_ERR_ARG;
}

/* A-init (PAPER.md:68-69 (2.9), "u = U0"):
 *   w_0 = phi,  w_{-1} = phi - (tau/2) psi   (reading A1; reduces to Algorithm 1's u = U0 for psi = 0). */
int oracle_wave2d_set_initial(oracle_wave2d_t *h, const double *phi, const double *psi, long ld)
{
    if (!h || !phi || ld < h->n1) return ORACLE_ERR_ARG;
    if (h->scheme == 1 && h->M < 1) return ORACLE_ERR_RANGE;
    for (int j = 0; j < h->n2; ++j)
        for (int i = 0; i < h->n1; ++i) {
            double p = phi[(long)j * ld + i];
            double q = psi ? psi[(long)j * ld + i] : 0.0;
            if (h->scheme == 0) {
                h->w[1][(size_t)j * h->n1 + i] = p;
                h->w[0][(size_t)j * h->n1 + i] = p - 0.5 * h->tau * q;
            } else {   /* (2.9) as printed: u^0 = phi, u^1 = u^0 + tau psi; the state is level k = 1 */
                h->w[0][(size_t)j * h->n1 + i] = p;
                h->w[1][(size_t)j * h->n1 + i] = p + h->tau * q;
            }
        }
    h->have_initial = 1;
    h->start_done = 0;
    h->n_done = h->scheme == 1 ? 2 : 0;
    return ORACLE_OK;
}

/* Second-order start of (2.8): u^1 += (tau^2 / 2) (c^0 Lap_h phi + g^0 s), with u^0 = phi in w[0], u^1 in w[1] and
 * Lap_h the five-point Laplacian with zero Dirichlet ghosts (2.10).  Applied at the first run: the speed and source
 * samples may be set after the initial data. */
static void oracle_second_order_start(oracle_wave2d_t *h)
{
    const double h1 = h->l / h->N1, h2 = h->l / h->N2, c0 = h->c_half[0], g0 = h->g_half ? h->g_half[0] : 1.0;
    const double *phi = h->w[0];
    for (int j = 0; j < h->n2; ++j)
        for (int i = 0; i < h->n1; ++i) {
            const size_t o = (size_t)j * h->n1 + i;
            const double we = i > 0 ? phi[o - 1] : 0.0, ea = i < h->n1 - 1 ? phi[o + 1] : 0.0;
            const double so = j > 0 ? phi[o - h->n1] : 0.0, no = j < h->n2 - 1 ? phi[o + h->n1] : 0.0;
            const double lap = (we - 2.0 * phi[o] + ea) / (h1 * h1) + (so - 2.0 * phi[o] + no) / (h2 * h2);
            h->w[1][o] += 0.5 * h->tau * h->tau * (c0 * lap + (h->s ? g0 * h->s[o] : 0.0));
        }
}

/* c_half[n] = c(n tau/2), n = 0..2M  (count == 2M+1), or one constant (count == 1). */
int oracle_wave2d_set_speed(oracle_wave2d_t *h, const double *c_half, int count)
{
    if (!h || !c_half || (count != 1 && count != 2 * h->M + 1)) return ORACLE_ERR_ARG;
    if (h->n_done > 0) return ORACLE_ERR_STATE;
    for (int n = 0; n < count; ++n) if (!(c_half[n] > 0.0)) return ORACLE_ERR_ARG;
    for (int n = 0; n <= 2 * h->M; ++n) h->c_half[n] = count == 1 ? c_half[0] : c_half[n];
    return ORACLE_OK;
}

/* Spatial speed factor: c(t,x,y) = c_half[n] * cs(x,y) (reading R16); cs NULL returns to c = c(t).  Scheme 0 only. */
int oracle_wave2d_set_speed_field(oracle_wave2d_t *h, const double *cs, long ld)
{
    if (!h) return ORACLE_ERR_ARG;
    if (h->n_done > (h->scheme == 1 ? 2 : 0)) return ORACLE_ERR_STATE;
    free(h->cs); h->cs = NULL;
    if (!cs) return ORACLE_OK;
    if (ld < h->n1 || h->scheme == 1) return ORACLE_ERR_ARG;
    for (int j = 0; j < h->n2; ++j)
        for (int i = 0; i < h->n1; ++i)
            if (!(cs[(long)j * ld + i] > 0.0)) return ORACLE_ERR_ARG;   /* PAPER.md:31, positive speed */
    h->cs = (double *)malloc(sizeof(double) * (size_t)h->n1 * (size_t)h->n2);
    if (!h->cs) return ORACLE_ERR_ALLOC;
    for (int j = 0; j < h->n2; ++j)
        memcpy(h->cs + (size_t)j * h->n1, cs + (long)j * ld, sizeof(double) * (size_t)h->n1);
    return ORACLE_OK;
}

/* f(t,x,y) = g(t) s(x,y); g_half[n] = g(n tau/2), n = 0..2M-1; g_half NULL means g == 1; s NULL clears. */
int oracle_wave2d_set_source(oracle_wave2d_t *h, const double *s, long ld, const double *g_half, int count)
{
    if (!h) return ORACLE_ERR_ARG;
    if (h->n_done > 0) return ORACLE_ERR_STATE;
    free(h->s); h->s = NULL; free(h->g_half); h->g_half = NULL;
    if (!s) return ORACLE_OK;
    if (ld < h->n1 || (g_half && count < 2 * h->M)) return ORACLE_ERR_ARG;
    h->s = (double *)malloc(sizeof(double) * (size_t)h->n1 * (size_t)h->n2);
    if (!h->s) return ORACLE_ERR_ALLOC;
    for (int j = 0; j < h->n2; ++j)
        memcpy(h->s + (size_t)j * h->n1, s + (long)j * ld, sizeof(double) * (size_t)h->n1);
    if (g_half) {
        h->g_half = (double *)malloc(sizeof(double) * (size_t)(2 * h->M > 0 ? 2 * h->M : 1));
        if (!h->g_half) return ORACLE_ERR_ALLOC;
        memcpy(h->g_half, g_half, sizeof(double) * (size_t)(2 * h->M));
    }
    return ORACLE_OK;
}

/* Algorithm 1's while-loop body, `steps` times: x half-step, y half-step, rotate. */
int oracle_wave2d_run(oracle_wave2d_t *h, int steps)
{
    if (!h || steps < 0) return ORACLE_ERR_ARG;
    if (!h->have_initial) return ORACLE_ERR_STATE;
    if (h->n_done / 2 + steps > h->M) return ORACLE_ERR_RANGE;
    if (h->scheme == 1 && (h->cs || h->sigma != 0.5)) return ORACLE_ERR_ARG;
    if (h->scheme == 0 && h->start != 1) return ORACLE_ERR_ARG;   /* (2.9) belongs to the three-level scheme (2.8) */
    if (h->scheme == 1 && h->start == 2 && !h->start_done && steps > 0) {
        if (h->n_done != 2) return ORACLE_ERR_STATE;
        oracle_second_order_start(h);
        h->start_done = 1;
    }
    if (h->scheme == 1) {   /* (2.8) factorised: level k -> k+1 needs c^{k-1}, c^{k+1}, g^k (integer levels) */
        for (int it = 0; it < steps; ++it) {
            const int k = h->n_done / 2;
            const double t2 = h->tau * h->tau, h1 = h->l / h->N1, h2 = h->l / h->N2;
            const double cp1 = h->c_half[2 * (k + 1)], cm1 = h->c_half[2 * (k - 1)];
            const double g = h->g_half ? h->g_half[2 * k] : 1.0;
            oracle_factored_step(h->n1, h->n2, t2 * cp1 / (2.0 * h1 * h1), t2 * cm1 / (2.0 * h1 * h1),
                                 t2 * cp1 / (2.0 * h2 * h2), t2 * cm1 / (2.0 * h2 * h2), t2 * g,
                                 h->w[0], h->w[1], h->s, h->w[2]);
            double *old = h->w[0];
            h->w[0] = h->w[1]; h->w[1] = h->w[2]; h->w[2] = old;
            h->n_done += 2;
        }
        return ORACLE_OK;
    }
    for (int it = 0; it < 2 * steps; ++it) {
        const int n = h->n_done;
        const int dir = n & 1;                                   /* x if n even, y if n odd */
        const double hd = h->l / (dir == 0 ? h->N1 : h->N2);     /* reading A3: h1 in x, h2 in y */
        const double t2 = h->tau * h->tau;
        const double ap = h->sigma * t2 * h->c_half[n + 1] / (hd * hd);                       /* sigma = 1/2: (2.11)-(2.12) */
        const double am = (1.0 - h->sigma) * t2 * h->c_half[n > 0 ? n - 1 : 0] / (hd * hd);   /* reading A5 */
        const double g = h->g_half ? h->g_half[n] : 1.0;                        /* reading A8 */
        const double q = h->kappa * t2 * g;
        if (h->cs) oracle_half_step_var(h->n1, h->n2, dir, ap, am, h->gamma, q, h->cs, h->w[0], h->w[1], h->s, h->w[2]);
        else oracle_half_step(h->n1, h->n2, dir, ap, am, h->gamma, q, h->w[0], h->w[1], h->s, h->w[2]);
        /* (w_prev, w_cur) <- (w_cur, w_next): "swap(u,Ux); swap(U0,Uy)" done one half-level at a time */
        double *old = h->w[0];
        h->w[0] = h->w[1]; h->w[1] = h->w[2]; h->w[2] = old;
        h->n_done = n + 1;
    }
    return ORACLE_OK;
}

static int copy_out(const oracle_wave2d_t *h, const double *src, double *dst, long ld)
{
    if (!h || !dst || ld < h->n1) return ORACLE_ERR_ARG;
    for (int j = 0; j < h->n2; ++j)
        memcpy(dst + (long)j * ld, src + (size_t)j * h->n1, sizeof(double) * (size_t)h->n1);
    return ORACLE_OK;
}

/* u^k (k = steps done) and u^{k-1/2} (scheme 1: u^{k-1}). */
int oracle_wave2d_get(const oracle_wave2d_t *h, double *u_out, long ld) { return h ? copy_out(h, h->w[1], u_out, ld) : ORACLE_ERR_ARG; }
int oracle_wave2d_get_prev(const oracle_wave2d_t *h, double *u_out, long ld) { return h ? copy_out(h, h->w[0], u_out, ld) : ORACLE_ERR_ARG; }
int oracle_wave2d_steps_done(const oracle_wave2d_t *h, int *k) { if (!h || !k) return ORACLE_ERR_ARG; *k = h->n_done / 2; return ORACLE_OK; }

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
