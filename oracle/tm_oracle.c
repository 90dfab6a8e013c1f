/*
 * tm_oracle.c -- plain, slow, double-precision CPU oracle for the Wilson twisted-mass
 * operator of arXiv 1311.4462.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call this file.  It shares no code with the CUDA path under
 * paper_1311_4462_b200/ and neither includes the other.
 *
 * What it computes (the plain definition, no even-odd tricks, no projector tricks, dense
 * 4x4 gamma matrices and dense 3x3 links on full-lattice lexicographic fields):
 *
 *   Eq. (2.1) [PAPER.md:50-52, equation itself lost in extraction; reading C1/C2]
 *       D = D_W (x) 1_f + i mu_bar gamma5 (x) tau3 + eps_bar 1 (x) tau1
 *     in the hopping-parameter normalisation  M = 2 kappa D = R - kappa D_hop,
 *       R = 1 + i a gamma5 tau3 + b tau1,  a = 2 kappa mu_bar,  b = 2 kappa eps_bar,
 *       R^{-1} = (1 - i a gamma5 tau3 - b tau1) / (1 + a^2 - b^2)          [PAPER.md:64 "R"]
 *   Hopping term [DESIGN.md reading C3; "hopping terms"]
 *       (D_hop psi)(x) = sum_mu  eta+_mu(x) (1 - gamma_mu) U_mu(x)        psi(x+mu)
 *                             +  eta-_mu(x) (1 + gamma_mu) U_mu(x-mu)^dag  psi(x-mu)
 *     periodic in space; in time eta = t_boundary on the wrapped hop, 1 elsewhere.
 *   gamma matrices [PAPER.md:52 "non-relativistic basis"; reading C5]
 *       gamma_k = [[0, i sigma_k], [-i sigma_k, 0]],  gamma_4 = diag(1,1,-1,-1),
 *       gamma_5 = gamma_1 gamma_2 gamma_3 gamma_4 (computed as that product here).
 *   Fused kernels [PAPER.md:68] and even-odd systems Eq. (2.2)-(2.4) [PAPER.md:60-66;
 *   DESIGN.md reading C4, C6, C7]:
 *       A      : out_p = R^{-1} (D_hop in)_p
 *       A-xpay : out_p = x_p - kappa^2 R^{-1} (D_hop in)_p
 *       B      : out_p = R x_p - kappa^2 (D_hop in)_p
 *       REC    : out_p = R^{-1} (x_p + kappa (D_hop in)_p)
 *       dagger : D_hop -> D_hop^dag (projectors swapped), R -> R^dag (a -> -a), same order.
 *
 * Parity status: pinned by tests/test_oracle_pins.py (P1-P12 of DESIGN.md).  Three pure
 * conventions are "parity unpinned" (no property of the paper fixes them; they are declared
 * in DESIGN.md): the sign of the eps_bar tau1 term, "1 - gamma_mu goes with the forward
 * hop", and the particular gamma_4-diagonal representation.
 *
 * Layouts (all C-contiguous, double, complex = (re, im)):
 *   spinor : [nf][V][4 spin][3 color]      V = X*Y*Z*T, lex = x1 + X*(x2 + Y*(x3 + Z*x4))
 *   gauge  : [4 mu][V][3 row][3 col]       U_mu(x) = link from x to x + mu_hat
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

enum { TMO_A = 0, TMO_A_XPAY = 1, TMO_B = 2, TMO_REC = 3 };
enum { TMO_ASYM = 0, TMO_SYM = 1 };

typedef struct {
    int X[4];            /* extents x1..x4 (x4 = time) */
    double kappa, mu, epsilon;
    int twist_flavor;    /* +1 / -1: single flavor with tau3 -> +-1 ; 0: non-degenerate doublet */
    int t_boundary;      /* -1 antiperiodic, +1 periodic in time */
} tmo_params;

int tmo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void tmo_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---- gamma matrices (reading C5) ------------------------------------------------------ */

static void pauli(int k, cplx s[2][2])
{
    memset(s, 0, 4 * sizeof(cplx));
    if (k == 0) { s[0][1] = 1; s[1][0] = 1; }
    if (k == 1) { s[0][1] = -I; s[1][0] = I; }
    if (k == 2) { s[0][0] = 1; s[1][1] = -1; }
}

/* idx 0..2: gamma_1..3 ; 3: gamma_4 ; 4: gamma_5 = gamma_1 gamma_2 gamma_3 gamma_4 */
static void gamma_mat(int idx, cplx g[4][4])
{
    memset(g, 0, 16 * sizeof(cplx));
    if (idx < 3) {
        cplx s[2][2];
        pauli(idx, s);
        for (int i = 0; i < 2; i++)
            for (int j = 0; j < 2; j++) {
                g[i][2 + j] = I * s[i][j];
                g[2 + i][j] = -I * s[i][j];
            }
    } else if (idx == 3) {
        g[0][0] = g[1][1] = 1;
        g[2][2] = g[3][3] = -1;
    } else {
        cplx acc[4][4], nxt[4][4], gm[4][4];
        gamma_mat(0, acc);
        for (int m = 1; m < 4; m++) {
            gamma_mat(m, gm);
            for (int i = 0; i < 4; i++)
                for (int j = 0; j < 4; j++) {
                    cplx s = 0;
                    for (int k = 0; k < 4; k++) s += acc[i][k] * gm[k][j];
                    nxt[i][j] = s;
                }
            memcpy(acc, nxt, sizeof(acc));
        }
        memcpy(g, acc, 16 * sizeof(cplx));
    }
}

void tmo_gamma(int idx, double *out /* [4][4][2] */)
{
    cplx g[4][4];
    gamma_mat(idx, g);
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            out[2 * (4 * i + j)] = creal(g[i][j]);
            out[2 * (4 * i + j) + 1] = cimag(g[i][j]);
        }
}

/* ---- lattice helpers --------------------------------------------------------------------- */

static long volume(const int X[4]) { return (long)X[0] * X[1] * X[2] * X[3]; }

static void coords(long lex, const int X[4], int x[4])
{
    for (int d = 0; d < 4; d++) { x[d] = (int)(lex % X[d]); lex /= X[d]; }
}

static long lexidx(const int x[4], const int X[4])
{
    return x[0] + (long)X[0] * (x[1] + (long)X[1] * (x[2] + (long)X[2] * x[3]));
}

int tmo_site_parity(long lex, const int *X)
{
    int x[4];
    coords(lex, X, x);
    return (x[0] + x[1] + x[2] + x[3]) & 1;
}

/* ---- hopping term at one site (reading C3) ------------------------------------------------ */

/* lexicographic index of the neighbour x + mu_hat (dir = 0) or x - mu_hat (dir = 1), periodic wrap */
static long neighbour(const int x[4], const int X[4], int mu, int dir)
{
    int y[4];
    memcpy(y, x, sizeof(y));
    y[mu] = (x[mu] + (dir ? -1 : 1) + X[mu]) % X[mu];
    return lexidx(y, X);
}

/* The hopping sum at `site`, given the spinor values nbv[2*mu + dir][f][s][c] already fetched from
 * the 8 neighbours (dir 0 = x + mu_hat, dir 1 = x - mu_hat):
 *   acc = sum_mu eta+ (1 - sgn gamma_mu) U_mu(x) psi(x+mu) + eta- (1 + sgn gamma_mu) U_mu(x-mu)^dag psi(x-mu)
 * sgn = +1 for D_hop, -1 for D_hop^dag (the two projectors swap). */
static void hop_from_neighbours(cplx acc[2][4][3], cplx nbv[8][2][4][3], const cplx *gauge,
                                const tmo_params *p, int nf, long site, int dagger)
{
    const long V = volume(p->X);
    int x[4];
    coords(site, p->X, x);
    for (int f = 0; f < nf; f++)
        for (int s = 0; s < 4; s++)
            for (int c = 0; c < 3; c++) acc[f][s][c] = 0;
    const double sgn = dagger ? -1.0 : 1.0;

    for (int mu = 0; mu < 4; mu++) {
        cplx g[4][4];
        gamma_mat(mu, g);

        /* forward hop: eta+ (1 - gamma_mu) U_mu(x) psi(x + mu) */
        double eta = (mu == 3 && x[3] == p->X[3] - 1) ? (double)p->t_boundary : 1.0;
        const cplx *U = gauge + ((long)mu * V + site) * 9;
        for (int f = 0; f < nf; f++) {
            cplx v[4][3];
            for (int s = 0; s < 4; s++)
                for (int c = 0; c < 3; c++) {
                    cplx t = 0;
                    for (int d = 0; d < 3; d++) t += U[3 * c + d] * nbv[2 * mu][f][s][d];
                    v[s][c] = t;
                }
            for (int s = 0; s < 4; s++)
                for (int c = 0; c < 3; c++) {
                    cplx t = 0;
                    for (int r = 0; r < 4; r++) t += ((s == r ? 1.0 : 0.0) - sgn * g[s][r]) * v[r][c];
                    acc[f][s][c] += eta * t;
                }
        }

        /* backward hop: eta- (1 + gamma_mu) U_mu(x - mu)^dag psi(x - mu) */
        eta = (mu == 3 && x[3] == 0) ? (double)p->t_boundary : 1.0;
        U = gauge + ((long)mu * V + neighbour(x, p->X, mu, 1)) * 9;
        for (int f = 0; f < nf; f++) {
            cplx v[4][3];
            for (int s = 0; s < 4; s++)
                for (int c = 0; c < 3; c++) {
                    cplx t = 0;
                    for (int d = 0; d < 3; d++) t += conj(U[3 * d + c]) * nbv[2 * mu + 1][f][s][d];
                    v[s][c] = t;
                }
            for (int s = 0; s < 4; s++)
                for (int c = 0; c < 3; c++) {
                    cplx t = 0;
                    for (int r = 0; r < 4; r++) t += ((s == r ? 1.0 : 0.0) + sgn * g[s][r]) * v[r][c];
                    acc[f][s][c] += eta * t;
                }
        }
    }
}

/* acc[f][s][c] = (D_hop in)(site) for dagger = 0, (D_hop^dag in)(site) for dagger = 1 */
static void hop_site(cplx acc[2][4][3], const cplx *in, const cplx *gauge, const tmo_params *p,
                     int nf, long site, int dagger)
{
    const long V = volume(p->X);
    int x[4];
    coords(site, p->X, x);
    cplx nbv[8][2][4][3];
    for (int mu = 0; mu < 4; mu++)
        for (int dir = 0; dir < 2; dir++) {
            long nb = neighbour(x, p->X, mu, dir);
            for (int f = 0; f < nf; f++)
                memcpy(nbv[2 * mu + dir][f], in + ((long)f * V + nb) * 12, 12 * sizeof(cplx));
        }
    hop_from_neighbours(acc, nbv, gauge, p, nf, site, dagger);
}

/* ---- local twist at one site (reading C2) -------------------------------------------------- */

/* out = R v (inverse = 0) or R^{-1} v (inverse = 1); dagger: a -> -a.  v, out: [nf][4][3].
 * Returns 0, or -1 if the inverse does not exist. */
static int twist_site(cplx out[2][4][3], cplx v[2][4][3], const tmo_params *p, int nf, int inverse,
                      int dagger)
{
    cplx g5[4][4];
    gamma_mat(4, g5);
    double a = 2.0 * p->kappa * p->mu;
    double b = 2.0 * p->kappa * p->epsilon;
    if (dagger) a = -a;
    double tau3[2] = { 1.0, -1.0 };
    if (nf == 1) { tau3[0] = (double)p->twist_flavor; b = 0.0; }
    double sg = inverse ? -1.0 : 1.0;   /* R^{-1} = (1 - i a g5 tau3 - b tau1) / (1 + a^2 - b^2) */
    double den = 1.0;
    if (inverse) {
        den = 1.0 + a * a - b * b;
        if (fabs(den) < 1e-12) return -1;
    }
    for (int f = 0; f < nf; f++)
        for (int s = 0; s < 4; s++)
            for (int c = 0; c < 3; c++) {
                cplx t = v[f][s][c];
                cplx g5v = 0;
                for (int r = 0; r < 4; r++) g5v += g5[s][r] * v[f][r][c];
                t += sg * I * a * tau3[f] * g5v;
                if (nf == 2) t += sg * b * v[1 - f][s][c];
                out[f][s][c] = t / den;
            }
    return 0;
}

static void load_site(cplx v[2][4][3], const cplx *field, long V, int nf, long site)
{
    for (int f = 0; f < nf; f++) memcpy(v[f], field + ((long)f * V + site) * 12, 12 * sizeof(cplx));
}

static void store_site(cplx *field, cplx v[2][4][3], long V, int nf, long site)
{
    for (int f = 0; f < nf; f++) memcpy(field + ((long)f * V + site) * 12, v[f], 12 * sizeof(cplx));
}

static int nflavor(const tmo_params *p) { return p->twist_flavor == 0 ? 2 : 1; }

/* ---- full-lattice operators ---------------------------------------------------------------- */

/* out = D_hop in (or D_hop^dag in) on every site */
int tmo_dhop(double *out_, const double *in_, const double *gauge_, const tmo_params *p, int dagger)
{
    cplx *out = (cplx *)out_;
    const cplx *in = (const cplx *)in_, *gauge = (const cplx *)gauge_;
    const long V = volume(p->X);
    const int nf = nflavor(p);
#pragma omp parallel for schedule(static)
    for (long site = 0; site < V; site++) {
        cplx acc[2][4][3];
        hop_site(acc, in, gauge, p, nf, site, dagger);
        store_site(out, acc, V, nf, site);
    }
    return 0;
}

/* out = R in or R^{-1} in on every site */
int tmo_twist(double *out_, const double *in_, const tmo_params *p, int inverse, int dagger)
{
    cplx *out = (cplx *)out_;
    const cplx *in = (const cplx *)in_;
    const long V = volume(p->X);
    const int nf = nflavor(p);
    int err = 0;
#pragma omp parallel for schedule(static)
    for (long site = 0; site < V; site++) {
        cplx v[2][4][3], w[2][4][3];
        load_site(v, in, V, nf, site);
        if (twist_site(w, v, p, nf, inverse, dagger)) {
#pragma omp atomic write
            err = -1;
        } else
            store_site(out, w, V, nf, site);
    }
    return err;
}

/* out = M in = (R - kappa D_hop) in  [= 2 kappa D of Eq. (2.1)]; dagger: R^dag - kappa D_hop^dag */
int tmo_mat(double *out_, const double *in_, const double *gauge_, const tmo_params *p, int dagger)
{
    cplx *out = (cplx *)out_;
    const cplx *in = (const cplx *)in_, *gauge = (const cplx *)gauge_;
    const long V = volume(p->X);
    const int nf = nflavor(p);
#pragma omp parallel for schedule(static)
    for (long site = 0; site < V; site++) {
        cplx acc[2][4][3], v[2][4][3], w[2][4][3];
        hop_site(acc, in, gauge, p, nf, site, dagger);
        load_site(v, in, V, nf, site);
        twist_site(w, v, p, nf, 0, dagger);
        for (int f = 0; f < nf; f++)
            for (int s = 0; s < 4; s++)
                for (int c = 0; c < 3; c++) w[f][s][c] -= p->kappa * acc[f][s][c];
        store_site(out, w, V, nf, site);
    }
    return 0;
}

/* ---- the fused kernels of PAPER.md:68 at one output site (reading C6) ---------------------- */

/* The local part: w = epilogue(acc, xv) for the four kernel types, acc = (D_hop in)(site). */
static int epilogue_site(cplx w[2][4][3], cplx acc[2][4][3], cplx xv[2][4][3], const tmo_params *p,
                         int nf, int dagger, int kernel_type)
{
    cplx t[2][4][3];
    const double k = p->kappa;
    int err = 0;
    switch (kernel_type) {
    case TMO_A:        /* R^{-1} D in */
        err = twist_site(w, acc, p, nf, 1, dagger);
        break;
    case TMO_A_XPAY:   /* x - kappa^2 R^{-1} D in */
        err = twist_site(t, acc, p, nf, 1, dagger);
        for (int f = 0; f < nf; f++)
            for (int s = 0; s < 4; s++)
                for (int c = 0; c < 3; c++) w[f][s][c] = xv[f][s][c] - k * k * t[f][s][c];
        break;
    case TMO_B:        /* R x - kappa^2 D in */
        err = twist_site(t, xv, p, nf, 0, dagger);
        for (int f = 0; f < nf; f++)
            for (int s = 0; s < 4; s++)
                for (int c = 0; c < 3; c++) w[f][s][c] = t[f][s][c] - k * k * acc[f][s][c];
        break;
    case TMO_REC:      /* R^{-1} (x + kappa D in) */
        for (int f = 0; f < nf; f++)
            for (int s = 0; s < 4; s++)
                for (int c = 0; c < 3; c++) t[f][s][c] = xv[f][s][c] + k * acc[f][s][c];
        err = twist_site(w, t, p, nf, 1, dagger);
        break;
    default:
        err = -2;
    }
    return err;
}

static int kernel_site(cplx w[2][4][3], const cplx *in, const cplx *x, const cplx *gauge,
                       const tmo_params *p, int nf, long site, int dagger, int kernel_type)
{
    const long V = volume(p->X);
    cplx acc[2][4][3], xv[2][4][3];
    hop_site(acc, in, gauge, p, nf, site, dagger);
    if (kernel_type != TMO_A) load_site(xv, x, V, nf, site);
    return epilogue_site(w, acc, xv, p, nf, dagger, kernel_type);
}

/* Full-lattice arrays; writes only the sites of `parity`; reads `in` only at parity 1-p
 * (D_hop connects opposite parities) and `x` only at parity p.  x may be NULL for A. */
int tmo_kernel(double *out_, const double *in_, const double *x_, const double *gauge_,
               const tmo_params *p, int parity, int dagger, int kernel_type)
{
    cplx *out = (cplx *)out_;
    const cplx *in = (const cplx *)in_, *x = (const cplx *)x_, *gauge = (const cplx *)gauge_;
    const long V = volume(p->X);
    const int nf = nflavor(p);
    if (kernel_type != TMO_A && !x) return -3;
    int err = 0;
#pragma omp parallel for schedule(static)
    for (long site = 0; site < V; site++) {
        if (tmo_site_parity(site, p->X) != parity) continue;
        cplx w[2][4][3];
        int e = kernel_site(w, in, x, gauge, p, nf, site, dagger, kernel_type);
        if (e) {
#pragma omp atomic write
            err = e;
        } else
            store_site(out, w, V, nf, site);
    }
    return err;
}

/* Same kernel, evaluated only at the listed output sites; out: [n][nf][4][3]. */
int tmo_kernel_sites(double *out_, const long *sites, long n, const double *in_, const double *x_,
                     const double *gauge_, const tmo_params *p, int dagger, int kernel_type)
{
    cplx *out = (cplx *)out_;
    const cplx *in = (const cplx *)in_, *x = (const cplx *)x_, *gauge = (const cplx *)gauge_;
    const int nf = nflavor(p);
    if (kernel_type != TMO_A && !x) return -3;
    int err = 0;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; i++) {
        cplx w[2][4][3];
        int e = kernel_site(w, in, x, gauge, p, nf, sites[i], dagger, kernel_type);
        if (e) {
#pragma omp atomic write
            err = e;
        }
        for (int f = 0; f < nf; f++) memcpy(out + ((long)i * nf + f) * 12, w[f], 12 * sizeof(cplx));
    }
    return err;
}

/* ---- composites: LHS of Eq. (2.2) / (2.3), and Eq. (2.4)  [PAPER.md:60-66] ------------------ */

/* out_e = M^_asym in_e = (R_ee - kappa^2 D_eo R_oo^{-1} D_oe) in_e           (type = ASYM)
 * out_e = M^_sym  in_e = (1    - kappa^2 R_ee^{-1} D_eo R_oo^{-1} D_oe) in_e  (type = SYM)
 * dagger = 1: the same two launches with the daggered kernels (reading C7).
 * Full-lattice arrays; only even sites of in are read and only even sites of out written. */
int tmo_matpc(double *out, const double *in, const double *gauge, const tmo_params *p, int type,
              int dagger)
{
    const long V = volume(p->X);
    const int nf = nflavor(p);
    double *tmp = (double *)calloc((size_t)V * nf * 24, sizeof(double));
    if (!tmp) return -4;
    int err = tmo_kernel(tmp, in, NULL, gauge, p, 1, dagger, TMO_A);          /* tmp_o = R^-1 D_oe in_e */
    if (!err)
        err = tmo_kernel(out, tmp, in, gauge, p, 0, dagger, type == TMO_ASYM ? TMO_B : TMO_A_XPAY);
    free(tmp);
    return err;
}

/* Eq. (2.4) (reading C4): psi_o = R_oo^{-1} (b_o + kappa D_oe psi_e).  Writes odd sites of out. */
int tmo_reconstruct_odd(double *out, const double *psi_e, const double *b_o, const double *gauge,
                        const tmo_params *p)
{
    return tmo_kernel(out, psi_e, b_o, gauge, p, 1, 0, TMO_REC);
}

/* Composite at the listed EVEN output sites only (sampled parity checks on big lattices, where a
 * full-lattice temporary is too slow): kernel A is evaluated at the 8 odd neighbours of each
 * sample, and the second kernel takes its hopping sum from those 8 values.  out: [n][nf][4][3]. */
int tmo_matpc_sites(double *out_, const long *sites, long n, const double *in_, const double *gauge_,
                    const tmo_params *p, int type, int dagger)
{
    cplx *out = (cplx *)out_;
    const cplx *in = (const cplx *)in_, *gauge = (const cplx *)gauge_;
    const long V = volume(p->X);
    const int nf = nflavor(p);
    int err = 0;
#pragma omp parallel for schedule(dynamic, 4)
    for (long i = 0; i < n; i++) {
        int x[4];
        coords(sites[i], p->X, x);
        cplx tmpv[8][2][4][3], acc[2][4][3], xv[2][4][3], w[2][4][3];
        int e = 0;
        for (int mu = 0; mu < 4; mu++)
            for (int dir = 0; dir < 2; dir++)     /* tmp_o = R_oo^-1 D_oe in_e at the neighbour */
                e |= kernel_site(tmpv[2 * mu + dir], in, NULL, gauge, p, nf, neighbour(x, p->X, mu, dir),
                                 dagger, TMO_A);
        hop_from_neighbours(acc, tmpv, gauge, p, nf, sites[i], dagger);
        load_site(xv, in, V, nf, sites[i]);
        e |= epilogue_site(w, acc, xv, p, nf, dagger, type == TMO_ASYM ? TMO_B : TMO_A_XPAY);
        for (int f = 0; f < nf; f++) memcpy(out + ((long)i * nf + f) * 12, w[f], 12 * sizeof(cplx));
        if (e) {
#pragma omp atomic write
            err = e;
        }
    }
    return err;
}
