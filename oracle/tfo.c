/*
 * oracle/tfo.c -- CPU ORACLE for the thin-film ADI step.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, fp64 restatement of the numerical method of
 *   Lam, Cummings, Kondic, "Computing dynamics of thin films via large scale
 *   GPU-based simulations" (arXiv:1806.10550), section 2 and App. A.
 * It shares NO code with the CUDA path (paper_1806_10550_b200/csrc).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call it.  Every function cites the passage it follows.  Readings of garbled or
 * ambiguous passages are the ones listed in DESIGN.md ("Readings", R1..R18).
 *
 * Conventions: field h[j*nx + i], i in [0,nx) along x (contiguous), j in [0,ny)
 * along y; cell centre (x_i,y_j) = ((i+1/2)dx,(j+1/2)dy)  (PAPER.md:173-179,
 * eqs (2.9)-(2.10)); s = dt/2.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): dense LU (penta solver), dense
 * 13-point Crank-Nicolson solve of the linear model (1.6), finite-difference
 * Jacobian, column sums, mass conservation, dispersion relation (1.4), dt-halving
 * order, G(u)=0 at convergence, fixed point, transpose symmetry.
 * The NLC (1.8)-(1.9) and polymer (1.12) disjoining pressures are pinned by finite
 * differences of Pi(h) as the paper defines it, the finite-difference Jacobian, G(u) = 0 and the dispersion
 * relation (tests/test_oracle_models.py).  The order of the two sweeps in tfo_step ((2.19) before (2.20)) and the two
 * lines of reading R18 (a finite, non-positive iterate ends the step; a NaN ratio surfaces in the residual) are pinned
 * by O12 / O13 of tests/test_oracle_pins.py.  Parity unpinned: nothing in this file.
 *
 * The optional "#pragma omp parallel for" lines are no-ops unless compiled with
 * -fopenmp (second build, used only for the all-core timed baseline).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

enum { TFO_OK = 0, TFO_NOT_CONVERGED = 1, TFO_ERR_INVALID_ARG = -1,
       TFO_ERR_UNSUPPORTED = -2, TFO_ERR_ALLOC = -4, TFO_ERR_STATE = -5 };

typedef struct tfo_ctx {
    int nx, ny;
    double dx, dy;
    /* model: 0 = thin film (1.7) with power-law Pi (K-term of (1.8)); 1 = linear (1.6);
     *        2 = thin film (1.7) with Pi_NLC (1.8)-(1.9); 3 = thin film (1.7) with Pi_POL (1.12) */
    int model;
    double cap0, cap1;               /* models 2,3: f0 = cap0 h^3, f1 = cap1 h^3 Pi'(h)  (reading R19)      */
    double pk, pb, pn, pbeta, pw;    /* NLC: K, b, N, beta, w of (1.8)-(1.9), (1.11)                      */
    double qc, qa1, qa2, qd;         /* polymer: C, A_SiOx, A_Si, d of (1.12)-(1.13)                      */
    double kappa, hstar; int n, m;   /* Pi(h) = kappa[(hstar/h)^n - (hstar/h)^m]   */
    double c0, c1;                   /* linear model f0 = c0, f1 = c1  */
    double tol; int max_iter, fixed_iters;
    int have_state;
    double *u;                       /* u^n                                           */
    double *uk, *bn, *R, *w, *v;     /* Newton iterate, b^n, rhs, intermediates       */
    double *f0, *f1, *g0, *g1;       /* f0,f1,f0',f1' at cell centres                 */
    double *L;                       /* discrete Laplacian at cell centres            */
} tfo_ctx;

/* integer power by repeated multiplication (reading R12: n,m integers, no pow()) */
static double ipow(double x, int p) { double r = 1.0; for (int k = 0; k < p; ++k) r *= x; return r; }

/*
 * Nonlinear functions at one cell centre.  PAPER.md:84-91, eqs (1.7)-(1.8) with
 * the capillary prefactor = 1 (reading R1):
 *   f0 = h^3, f0' = 3h^2, f1 = h^3 Pi'(h), f1' = 3h^2 Pi'(h) + h^3 Pi''(h),
 *   Pi'(h)  = kappa[ m h*^m / h^(m+1) - n h*^n / h^(n+1) ],
 *   Pi''(h) = kappa[ n(n+1) h*^n / h^(n+2) - m(m+1) h*^m / h^(m+2) ].
 * Linear model (1.6): f0 = c0, f1 = c1, derivatives 0.
 */

#define TFO_PI 3.14159265358979323846

/* Pi(h) exactly as the paper defines it -- used by the pins to difference, never by the solver.
 *   NLC, (1.8)-(1.9):  Pi = K[(b/h)^3 - (b/h)^2] + (N/2) [m(h)/h]^2,
 *        m = g h^2/(h^2 + beta^2),  g = (1/2)[1 + tanh((h - 2b)/w)];
 *   polymer, (1.12):    Pi = -d psi/dh,  psi = C/h^8 - A1/(12 pi h^2) + (A1 - A2)/(12 pi (h+d)^2). */
static double pressure(const tfo_ctx *c, double h)
{
    if (c->model == 2) {
        double r = c->pb / h;
        double g = 0.5 * (1.0 + tanh((h - 2.0 * c->pb) / c->pw));
        double m = g * h * h / (h * h + c->pbeta * c->pbeta);
        return c->pk * (r * r * r - r * r) + 0.5 * c->pn * (m / h) * (m / h);
    }
    if (c->model == 3) {
        double hd = h + c->qd;
        return 8.0 * c->qc / pow(h, 9) - c->qa1 / (6.0 * TFO_PI * h * h * h) + (c->qa1 - c->qa2) / (6.0 * TFO_PI * hd * hd * hd);
    }
    double r = c->hstar / h;
    return c->kappa * (ipow(r, c->n) - ipow(r, c->m));
}

/* Pi'(h) and Pi''(h) of the NLC and polymer pressures, by the chain and quotient rules on the definitions above:
 *   NLC: with D = h^2 + beta^2, M = m/h = g h/D, x = (h - 2b)/w, t = tanh x:
 *        g' = (1 - t^2)/(2w),  g'' = -t (1 - t^2)/w^2,
 *        M' = g' h/D + g (beta^2 - h^2)/D^2,
 *        M'' = g'' h/D + 2 g' (beta^2 - h^2)/D^2 + g (2h^3 - 6 h beta^2)/D^3,
 *        Pi' = K[-3 b^3/h^4 + 2 b^2/h^3] + N M M',   Pi'' = K[12 b^3/h^5 - 6 b^2/h^4] + N (M'^2 + M M'');
 *   polymer: Pi' = -72 C/h^10 + A1/(2 pi h^4) - (A1 - A2)/(2 pi (h+d)^4),
 *            Pi'' = 720 C/h^11 - 2 A1/(pi h^5) + 2 (A1 - A2)/(pi (h+d)^5). */
static void pressure_derivatives(const tfo_ctx *c, double h, double *P1, double *P2)
{
    if (c->model == 2) {
        double b = c->pb, w = c->pw, be2 = c->pbeta * c->pbeta;
        double t = tanh((h - 2.0 * b) / w);
        double g = 0.5 * (1.0 + t), g1 = (1.0 - t * t) / (2.0 * w), g2 = -t * (1.0 - t * t) / (w * w);
        double D = h * h + be2;
        double M = g * h / D;
        double M1 = g1 * h / D + g * (be2 - h * h) / (D * D);
        double M2 = g2 * h / D + 2.0 * g1 * (be2 - h * h) / (D * D) + g * (2.0 * h * h * h - 6.0 * h * be2) / (D * D * D);
        double r = 1.0 / h;
        *P1 = c->pk * (-3.0 * b * b * b * ipow(r, 4) + 2.0 * b * b * ipow(r, 3)) + c->pn * M * M1;
        *P2 = c->pk * (12.0 * b * b * b * ipow(r, 5) - 6.0 * b * b * ipow(r, 4)) + c->pn * (M1 * M1 + M * M2);
        return;
    }
    double r = 1.0 / h, rd = 1.0 / (h + c->qd), da = c->qa1 - c->qa2;
    *P1 = -72.0 * c->qc * ipow(r, 10) + c->qa1 * ipow(r, 4) / (2.0 * TFO_PI) - da * ipow(rd, 4) / (2.0 * TFO_PI);
    *P2 = 720.0 * c->qc * ipow(r, 11) - 2.0 * c->qa1 * ipow(r, 5) / TFO_PI + 2.0 * da * ipow(rd, 5) / TFO_PI;
}

static void model_functions(const tfo_ctx *c, double h, double *f0, double *f1, double *g0, double *g1)
{
    if (c->model == 1) { *f0 = c->c0; *f1 = c->c1; *g0 = 0.0; *g1 = 0.0; return; }
    if (c->model >= 2) {
        /* (1.7), with caller-supplied prefactors (reading R19): f0 = cap0 h^3, f1 = cap1 h^3 Pi' */
        double P1, P2;
        pressure_derivatives(c, h, &P1, &P2);
        double h2 = h * h, h3 = h2 * h;
        *f0 = c->cap0 * h3; *g0 = c->cap0 * 3.0 * h2;
        *f1 = c->cap1 * h3 * P1; *g1 = c->cap1 * (3.0 * h2 * P1 + h3 * P2);
        return;
    }
    double r = 1.0 / h;
    double hn = ipow(c->hstar, c->n), hm = ipow(c->hstar, c->m);
    double P1 = c->kappa * (c->m * hm * ipow(r, c->m + 1) - c->n * hn * ipow(r, c->n + 1));
    double P2 = c->kappa * (c->n * (c->n + 1) * hn * ipow(r, c->n + 2)
                          - c->m * (c->m + 1) * hm * ipow(r, c->m + 2));
    double h2 = h * h, h3 = h2 * h;
    *f0 = h3; *g0 = 3.0 * h2;
    *f1 = h3 * P1; *g1 = 3.0 * h2 * P1 + h3 * P2;
}

/* ghost points by reflection about the boundary faces: u_n = u_nnn = 0,
 * PAPER.md:297-304, eq (2.28).  idx -1 -> 0, -2 -> 1, N -> N-1, N+1 -> N-2. */
static int refl(int k, int N) { if (k < 0) return -k - 1; if (k >= N) return 2 * N - 1 - k; return k; }

static double at(const double *h, int nx, int ny, int i, int j)
{ return h[(size_t)refl(j, ny) * nx + refl(i, nx)]; }

static void fill_functions(tfo_ctx *c, const double *h)
{
    size_t N = (size_t)c->nx * c->ny;
#pragma omp parallel for
    for (size_t p = 0; p < N; ++p) model_functions(c, h[p], &c->f0[p], &c->f1[p], &c->g0[p], &c->g1[p]);
}

/*
 * Full operator D(h).  PAPER.md:183 eq (2.11), 262-293 (2.23)-(2.27):
 *   D = (Fx,+ - Fx,-)/dx + (Fy,+ - Fy,-)/dy,   F = f0(h) d/ds(lap h) + f1(h) dh/ds  (2.1),
 * L = lap h from cell-centre values; f at a face = mean of the two adjacent
 * cell-centre values (2.27); the four boundary faces carry zero flux (2.28),
 * PAPER.md:302.  Needs c->f0,c->f1 filled for this h.
 */
static void operator_D(tfo_ctx *c, const double *h, double *D)
{
    const int nx = c->nx, ny = c->ny; const double dx = c->dx, dy = c->dy;
#pragma omp parallel for
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i)
            c->L[(size_t)j * nx + i] =
                (at(h, nx, ny, i + 1, j) - 2.0 * at(h, nx, ny, i, j) + at(h, nx, ny, i - 1, j)) / (dx * dx)
              + (at(h, nx, ny, i, j + 1) - 2.0 * at(h, nx, ny, i, j) + at(h, nx, ny, i, j - 1)) / (dy * dy);
#pragma omp parallel for
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            size_t p = (size_t)j * nx + i;
            double Fxp = 0.0, Fxm = 0.0, Fyp = 0.0, Fym = 0.0;
            if (i + 1 < nx) { size_t q = p + 1;
                Fxp = 0.5 * (c->f0[p] + c->f0[q]) * (c->L[q] - c->L[p]) / dx
                    + 0.5 * (c->f1[p] + c->f1[q]) * (h[q] - h[p]) / dx; }
            if (i > 0) { size_t q = p - 1;
                Fxm = 0.5 * (c->f0[q] + c->f0[p]) * (c->L[p] - c->L[q]) / dx
                    + 0.5 * (c->f1[q] + c->f1[p]) * (h[p] - h[q]) / dx; }
            if (j + 1 < ny) { size_t q = p + nx;
                Fyp = 0.5 * (c->f0[p] + c->f0[q]) * (c->L[q] - c->L[p]) / dy
                    + 0.5 * (c->f1[p] + c->f1[q]) * (h[q] - h[p]) / dy; }
            if (j > 0) { size_t q = p - nx;
                Fym = 0.5 * (c->f0[q] + c->f0[p]) * (c->L[p] - c->L[q]) / dy
                    + 0.5 * (c->f1[q] + c->f1[p]) * (h[p] - h[q]) / dy; }
            D[p] = (Fxp - Fxm) / dx + (Fyp - Fym) / dy;
        }
}

/*
 * Pure-direction Jacobian bands of one line.  PAPER.md:274-278, eq (2.26): J_s is the
 * Jacobian of (F_{s,+} - F_{s,-})/ds where F "only contains derivatives with respect
 * to its subscript"; PAPER.md:748 (B_i needs x-neighbours only).  Reading R5.
 * Line values h_0..h_{N-1} (with f0,f1,f0',f1' at the same points), spacing d.
 * Interior face k+1/2 (0 <= k <= N-2):
 *   T = (h_{k+2} - 3h_{k+1} + 3h_k - h_{k-1})/d^3,  G = (h_{k+1} - h_k)/d   (ghosts reflected),
 *   F = fb0*T + fb1*G,  fb = mean of the two cell values (2.27),
 *   dF/dh_{k-1} = -fb0/d^3
 *   dF/dh_k     =  3fb0/d^3 - fb1/d + f0'_k/2 * T + f1'_k/2 * G
 *   dF/dh_{k+1} = -3fb0/d^3 + fb1/d + f0'_{k+1}/2 * T + f1'_{k+1}/2 * G
 *   dF/dh_{k+2} =  fb0/d^3.
 * Implicit stencil folded at the boundaries: ghost h_{-1} == h_0 so
 * dF/dh_{-1} is added to dF/dh_0; ghost h_N == h_{N-1} likewise.  Boundary faces: 0.
 * Row i of J = (dF_{i+1/2} - dF_{i-1/2})/d -> bands e,c,q,a,b on columns i-2..i+2.
 * `stride` lets the same routine walk a row (1) or a column (nx) of the 2-D arrays.
 */
static void jacobian_bands_line(int N, double d, size_t stride,
                                const double *h, const double *f0, const double *f1,
                                const double *g0, const double *g1,
                                double *e, double *cc, double *q, double *a, double *b)
{
    double *P = (double *)calloc((size_t)4 * (N + 1), sizeof(double)); /* P[4*(k+1)+t], face k=-1..N-1 */
    const double d3 = d * d * d;
    for (int k = 0; k <= N - 2; ++k) {
        double hm1 = h[(size_t)refl(k - 1, N) * stride], h0 = h[(size_t)k * stride];
        double h1 = h[(size_t)(k + 1) * stride], h2 = h[(size_t)refl(k + 2, N) * stride];
        double fb0 = 0.5 * (f0[(size_t)k * stride] + f0[(size_t)(k + 1) * stride]);
        double fb1 = 0.5 * (f1[(size_t)k * stride] + f1[(size_t)(k + 1) * stride]);
        double T = (h2 - 3.0 * h1 + 3.0 * h0 - hm1) / d3, G = (h1 - h0) / d;
        double *p = P + 4 * (k + 1);
        p[0] = -fb0 / d3;
        p[1] = 3.0 * fb0 / d3 - fb1 / d + 0.5 * g0[(size_t)k * stride] * T + 0.5 * g1[(size_t)k * stride] * G;
        p[2] = -3.0 * fb0 / d3 + fb1 / d + 0.5 * g0[(size_t)(k + 1) * stride] * T + 0.5 * g1[(size_t)(k + 1) * stride] * G;
        p[3] = fb0 / d3;
        if (k - 1 < 0) { p[1] += p[0]; p[0] = 0.0; }
        if (k + 2 >= N) { p[2] += p[3]; p[3] = 0.0; }
    }
    for (int i = 0; i < N; ++i) {
        const double *pp = P + 4 * (i + 1);   /* face i+1/2 (k = i);  zero if i = N-1 */
        const double *pm = P + 4 * i;         /* face i-1/2 (k = i-1); zero if i = 0  */
        e[i]  = (-pm[0]) / d;
        cc[i] = (pp[0] - pm[1]) / d;
        q[i]  = (pp[1] - pm[2]) / d;
        a[i]  = (pp[2] - pm[3]) / d;
        b[i]  = (pp[3]) / d;
    }
    free(P);
}

/*
 * Pentadiagonal solve, LU without pivoting (eq (A.5)):
 * row i:  e_i x_{i-2} + c_i x_{i-1} + d_i x_i + a_i x_{i+1} + b_i x_{i+2} = y_i.
 * Entries that fall outside the matrix (e_0,e_1,c_0,a_{N-1},b_{N-2},b_{N-1}) are ignored.
 * Forward (L z' = y folded with the U scaling):  gamma_i = c_i - alpha_{i-2} e_i,
 *   mu_i = d_i - beta_{i-2} e_i - alpha_{i-1} gamma_i,  alpha_i = (a_i - beta_{i-1} gamma_i)/mu_i,
 *   beta_i = b_i/mu_i,  z_i = (y_i - z_{i-2} e_i - z_{i-1} gamma_i)/mu_i.
 * Backward: x_i = z_i - alpha_i x_{i+1} - beta_i x_{i+2}.
 * Bands are walked with stride sb, y and x with stride sv.
 */
static void penta_solve_line(int N, size_t sb, size_t sv, const double *e, const double *c, const double *d,
                             const double *a, const double *b, const double *y, double *x,
                             double *al, double *be, double *z /* scratch, length N, unit stride */)
{
    for (int i = 0; i < N; ++i) {
        double ei = (i >= 2) ? e[i * sb] : 0.0, ci = (i >= 1) ? c[i * sb] : 0.0;
        double ai = (i <= N - 2) ? a[i * sb] : 0.0, bi = (i <= N - 3) ? b[i * sb] : 0.0;
        double al2 = (i >= 2) ? al[i - 2] : 0.0, be2 = (i >= 2) ? be[i - 2] : 0.0, z2 = (i >= 2) ? z[i - 2] : 0.0;
        double al1 = (i >= 1) ? al[i - 1] : 0.0, be1 = (i >= 1) ? be[i - 1] : 0.0, z1 = (i >= 1) ? z[i - 1] : 0.0;
        double gam = ci - al2 * ei;
        double mu = d[i * sb] - be2 * ei - al1 * gam;
        al[i] = (ai - be1 * gam) / mu;
        be[i] = bi / mu;
        z[i] = (y[i * sv] - z2 * ei - z1 * gam) / mu;
    }
    for (int i = N - 1; i >= 0; --i) {
        double x1 = (i + 1 < N) ? x[(size_t)(i + 1) * sv] : 0.0, x2 = (i + 2 < N) ? x[(size_t)(i + 2) * sv] : 0.0;
        x[(size_t)i * sv] = z[i] - al[i] * x1 - be[i] * x2;
    }
}

/* Solve (I + s J_dir(uk)) out = rhs for every line of direction dir (0: x rows, 1: y columns).
 * PAPER.md:232-234 eqs (2.19)-(2.20); (A.1)-(A.2),(A.4) PAPER.md:697-712. */
static void directional_solve(tfo_ctx *c, int dir, double s, const double *uk, const double *rhs, double *out)
{
    const int nx = c->nx, ny = c->ny;
    const int nlines = dir ? nx : ny, N = dir ? ny : nx;
    const size_t st = dir ? (size_t)nx : 1;
    const double d = dir ? c->dy : c->dx;
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * 8 * (size_t)N);
        double *e = buf, *cc = buf + N, *q = buf + 2 * N, *a = buf + 3 * N, *b = buf + 4 * N;
        double *al = buf + 5 * N, *be = buf + 6 * N, *z = buf + 7 * N;
#pragma omp for
        for (int l = 0; l < nlines; ++l) {
            size_t off = dir ? (size_t)l : (size_t)l * nx;
            jacobian_bands_line(N, d, st, uk + off, c->f0 + off, c->f1 + off, c->g0 + off, c->g1 + off, e, cc, q, a, b);
            for (int i = 0; i < N; ++i) { e[i] *= s; cc[i] *= s; q[i] = 1.0 + s * q[i]; a[i] *= s; b[i] *= s; }
            penta_solve_line(N, 1, st, e, cc, q, a, b, rhs + off, out + off, al, be, z);
        }
        free(buf);
    }
}

/* ------------------------------------------------------------------ public C-ABI (tfo_*) */

static int alloc_fields(tfo_ctx *c)
{
    size_t N = (size_t)c->nx * c->ny;
    double **f[] = { &c->u, &c->uk, &c->bn, &c->R, &c->w, &c->v, &c->f0, &c->f1, &c->g0, &c->g1, &c->L };
    for (size_t k = 0; k < sizeof(f) / sizeof(f[0]); ++k) {
        *f[k] = (double *)calloc(N, sizeof(double));
        if (!*f[k]) return TFO_ERR_ALLOC;
    }
    return TFO_OK;
}

/* Problem statement: PAPER.md:47 (1.1), 86-91 (1.7)-(1.8), 297-302 (2.28).  bc must be 0 (no-flux). */
int tfo_create(tfo_ctx **out, int nx, int ny, double dx, double dy,
               double kappa, double hstar, int n, int m, int bc)
{
    if (!out) return TFO_ERR_INVALID_ARG;
    *out = NULL;
    if (nx < 5 || ny < 5 || !(dx > 0) || !(dy > 0) || !(kappa > 0) || !(hstar > 0) || m < 1 || n <= m)
        return TFO_ERR_INVALID_ARG;
    if (bc != 0) return TFO_ERR_UNSUPPORTED;
    tfo_ctx *c = (tfo_ctx *)calloc(1, sizeof(tfo_ctx));
    if (!c) return TFO_ERR_ALLOC;
    c->nx = nx; c->ny = ny; c->dx = dx; c->dy = dy;
    c->model = 0; c->kappa = kappa; c->hstar = hstar; c->n = n; c->m = m;
    c->tol = 1e-10; c->max_iter = 10; c->fixed_iters = 0;   /* K = 10: PAPER.md:250 */
    int rc = alloc_fields(c);
    if (rc != TFO_OK) return rc;
    *out = c;
    return TFO_OK;
}

/* Switch to the linear test model (1.6): f0 = c0, f1 = c1. Oracle-only (pins O4/O5). */
int tfo_set_model_linear(tfo_ctx *c, double c0, double c1)
{ if (!c) return TFO_ERR_INVALID_ARG; c->model = 1; c->c0 = c0; c->c1 = c1; return TFO_OK; }

/* Disjoining pressure of SURVEY.md 8(f) row f-1.  kind 2: NLC, p = {cap0, cap1, K, b, N, beta, w};
 * kind 3: polymer, p = {cap0, cap1, C, A_SiOx, A_Si, d}. */
int tfo_set_pressure(tfo_ctx *c, int kind, const double *p, int np)
{
    if (!c || !p) return TFO_ERR_INVALID_ARG;
    if (kind == 2 && np == 7) {
        c->cap0 = p[0]; c->cap1 = p[1]; c->pk = p[2]; c->pb = p[3]; c->pn = p[4]; c->pbeta = p[5]; c->pw = p[6];
        if (!(c->pb > 0) || !(c->pw > 0)) return TFO_ERR_INVALID_ARG;
    } else if (kind == 3 && np == 6) {
        c->cap0 = p[0]; c->cap1 = p[1]; c->qc = p[2]; c->qa1 = p[3]; c->qa2 = p[4]; c->qd = p[5];
        if (!(c->qd > 0)) return TFO_ERR_INVALID_ARG;
    } else return TFO_ERR_INVALID_ARG;
    if (!(c->cap0 > 0) || !(c->cap1 > 0)) return TFO_ERR_INVALID_ARG;
    c->model = kind;
    return TFO_OK;
}

/* pins only: Pi(h) as defined by the paper, and the four cell functions, at n points */
int tfo_pressure(tfo_ctx *c, int n, const double *h, double *Pi)
{ if (!c || !h || !Pi) return TFO_ERR_INVALID_ARG; for (int k = 0; k < n; ++k) Pi[k] = pressure(c, h[k]); return TFO_OK; }
int tfo_cell_functions(tfo_ctx *c, int n, const double *h, double *f0, double *f1, double *g0, double *g1)
{
    if (!c || !h || !f0 || !f1 || !g0 || !g1) return TFO_ERR_INVALID_ARG;
    for (int k = 0; k < n; ++k) model_functions(c, h[k], f0 + k, f1 + k, g0 + k, g1 + k);
    return TFO_OK;
}

int tfo_set_newton(tfo_ctx *c, double tol, int max_iter, int fixed_iters)
{
    if (!c || !(tol >= 1e-14) || max_iter < 1 || fixed_iters < 0) return TFO_ERR_INVALID_ARG;
    c->tol = tol; c->max_iter = max_iter; c->fixed_iters = fixed_iters;
    return TFO_OK;
}

int tfo_set_state(tfo_ctx *c, const double *h)
{
    if (!c || !h) return TFO_ERR_INVALID_ARG;
    size_t N = (size_t)c->nx * c->ny;
    for (size_t p = 0; p < N; ++p)
        if (!isfinite(h[p]) || (c->model != 1 && !(h[p] > 0))) return TFO_ERR_INVALID_ARG;
    memcpy(c->u, h, N * sizeof(double));
    c->have_state = 1;
    return TFO_OK;
}

int tfo_get_state(tfo_ctx *c, double *h)
{
    if (!c || !h) return TFO_ERR_INVALID_ARG;
    if (!c->have_state) return TFO_ERR_STATE;
    memcpy(h, c->u, (size_t)c->nx * c->ny * sizeof(double));
    return TFO_OK;
}

/*
 * One time step.  PAPER.md:199 (2.14), 207 (2.15), 232-237 (2.19)-(2.21), 243-248 (2.22), 719:
 *   b^n = u^n - s D(u^n);  u_(0) = u^n;
 *   repeat: R = b^n - u_(k) - s D(u_(k));  (I + s J_y) w = R;  (I + s J_x) v = w;
 *           res = max |v/u_(k)|;  u_(k+1) = u_(k) + v;
 *   accept when res < tol; reject (state stays u^n) after max_iter iterations or when
 *   an iterate is not finite / not positive (reading R18).  With fixed_iters = K > 0:
 *   exactly K iterations, accepted unless one of the K iterates was not finite / not
 *   positive (R18 again: such a field is not a state).  Sweep order y then x (R3).
 */
int tfo_step(tfo_ctx *c, double dt, int *newton_iters, double *residual)
{
    if (!c || !(dt > 0)) return TFO_ERR_INVALID_ARG;
    if (!c->have_state) return TFO_ERR_STATE;
    const size_t N = (size_t)c->nx * c->ny;
    const double s = 0.5 * dt;
    fill_functions(c, c->u);
    operator_D(c, c->u, c->R);
    for (size_t p = 0; p < N; ++p) c->bn[p] = c->u[p] - s * c->R[p];
    memcpy(c->uk, c->u, N * sizeof(double));
    const int kmax = c->fixed_iters > 0 ? c->fixed_iters : c->max_iter;
    int k = 0, status = TFO_NOT_CONVERGED, anybad = 0; double res = 0.0;
    while (k < kmax) {
        fill_functions(c, c->uk);
        operator_D(c, c->uk, c->R);
        for (size_t p = 0; p < N; ++p) c->R[p] = c->bn[p] - c->uk[p] - s * c->R[p];
        directional_solve(c, 1, s, c->uk, c->R, c->w);     /* (2.19): implicit y */
        directional_solve(c, 0, s, c->uk, c->w, c->v);     /* (2.20): implicit x */
        res = 0.0; int bad = 0;
        for (size_t p = 0; p < N; ++p) {
            double r = fabs(c->v[p] / c->uk[p]);           /* (2.22), denominator u_(k) */
            if (!(r <= res)) res = r;                      /* NaN propagates into res   */
            c->uk[p] += c->v[p];                           /* (2.21) */
            if (!isfinite(c->uk[p]) || (c->model != 1 && !(c->uk[p] > 0))) bad = 1;
        }
        ++k;
        if (bad || res != res) anybad = 1;
        if (c->fixed_iters > 0) { if (k == kmax && !anybad) status = TFO_OK; continue; }
        if (bad) break;
        if (res < c->tol) { status = TFO_OK; break; }
    }
    if (status == TFO_OK) memcpy(c->u, c->uk, N * sizeof(double));
    if (newton_iters) *newton_iters = k;
    if (residual) *residual = res;
    return status;
}

/* Mass dx*dy*sum(h) (PAPER.md:352 (3.2) times the domain area), pairwise summation. */
static double pairwise_sum(const double *x, size_t n)
{
    if (n <= 8) { double s = 0.0; for (size_t k = 0; k < n; ++k) s += x[k]; return s; }
    size_t h = n / 2; return pairwise_sum(x, h) + pairwise_sum(x + h, n - h);
}
int tfo_mass(tfo_ctx *c, double *mass)
{
    if (!c || !mass) return TFO_ERR_INVALID_ARG;
    if (!c->have_state) return TFO_ERR_STATE;
    *mass = c->dx * c->dy * pairwise_sum(c->u, (size_t)c->nx * c->ny);
    return TFO_OK;
}

void tfo_destroy(tfo_ctx *c)
{
    if (!c) return;
    double *f[] = { c->u, c->uk, c->bn, c->R, c->w, c->v, c->f0, c->f1, c->g0, c->g1, c->L };
    for (size_t k = 0; k < sizeof(f) / sizeof(f[0]); ++k) free(f[k]);
    free(c);
}

/* ---- pieces exposed for the pins and for per-kernel parity ---- */

/* D(h) of (2.11)/(2.25) for an arbitrary field h (nx*ny). */
int tfo_operator_D(tfo_ctx *c, const double *h, double *D)
{
    if (!c || !h || !D) return TFO_ERR_INVALID_ARG;
    fill_functions(c, h); operator_D(c, h, D); return TFO_OK;
}

/* Bands of J_dir(h) (NOT I + sJ) for every line, each output nx*ny in field layout:
 * band value of row (i,j) stored at [j*nx+i].  dir 0: x, 1: y. */
int tfo_jacobian_bands(tfo_ctx *c, int dir, const double *h, double *e, double *cc, double *q, double *a, double *b)
{
    if (!c || !h) return TFO_ERR_INVALID_ARG;
    fill_functions(c, h);
    const int nx = c->nx, ny = c->ny, nl = dir ? nx : ny, N = dir ? ny : nx;
    const size_t st = dir ? (size_t)nx : 1; const double d = dir ? c->dy : c->dx;
    double *buf = (double *)malloc(sizeof(double) * 5 * (size_t)N);
    for (int l = 0; l < nl; ++l) {
        size_t off = dir ? (size_t)l : (size_t)l * nx;
        jacobian_bands_line(N, d, st, h + off, c->f0 + off, c->f1 + off, c->g0 + off, c->g1 + off,
                            buf, buf + N, buf + 2 * N, buf + 3 * N, buf + 4 * N);
        for (int i = 0; i < N; ++i) {
            e[off + i * st] = buf[i]; cc[off + i * st] = buf[N + i]; q[off + i * st] = buf[2 * N + i];
            a[off + i * st] = buf[3 * N + i]; b[off + i * st] = buf[4 * N + i];
        }
    }
    free(buf);
    return TFO_OK;
}

/* One Newton half: out = (I + s J_dir(uk))^{-1} rhs  for all lines. */
int tfo_directional_solve(tfo_ctx *c, int dir, double s, const double *uk, const double *rhs, double *out)
{
    if (!c || !uk || !rhs || !out) return TFO_ERR_INVALID_ARG;
    fill_functions(c, uk); directional_solve(c, dir, s, uk, rhs, out); return TFO_OK;
}

/*
 * Batched pentadiagonal solve (BASELINE.json config 4).  Six arrays in the 2-D layout
 * [nrow][ncol] row-major.  dir 0: system s = row s (contiguous, nsys = nrow, len = ncol);
 * dir 1: system s = column s (strided, nsys = ncol, len = nrow).  Host pointers.
 */
int tfo_penta_solve(int nrow, int ncol, int dir, const double *e, const double *c, const double *d,
                    const double *a, const double *b, const double *rhs, double *x)
{
    if (nrow < 1 || ncol < 1 || !e || !c || !d || !a || !b || !rhs || !x) return TFO_ERR_INVALID_ARG;
    const int nsys = dir ? ncol : nrow, len = dir ? nrow : ncol;
    const size_t st = dir ? (size_t)ncol : 1;
    if (len < 3) return TFO_ERR_INVALID_ARG;
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * 3 * (size_t)len);
#pragma omp for
        for (int l = 0; l < nsys; ++l) {
            size_t off = dir ? (size_t)l : (size_t)l * ncol;
            penta_solve_line(len, st, st, e + off, c + off, d + off, a + off, b + off, rhs + off, x + off,
                             buf, buf + len, buf + 2 * len);
        }
        free(buf);
    }
    return TFO_OK;
}

int tfo_num_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
