/*
 * pb_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU implementation (fp64, O(N^2) loops) of the discretisation "D0" of
 * the multi-surface boundary-element Poisson-Boltzmann operator of PyGBe (arXiv:1309.4018), written
 * from /root/reference/PAPER.md.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.  It shares no code, header, table or constant with the CUDA path.
 *
 * Every function cites the passage of PAPER.md it follows (":line", section / equation).  Readings of
 * silent or garbled passages are those listed in DESIGN.md ("Readings", A1..A20).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): paper's -41.2465 kJ/mol (:229), Born-with-salt and
 * Kirkwood closed forms, Gauss identity (-1/2, -1, 0), concentric Stern / cavity analytic solutions,
 * quadrature moment exactness, closed-form 1/r self integral.
 * Parity unpinned: the GMRES iterate path (oracle/gmres.py) -- only residuals and energies are pinned.
 *
 * Layout conventions (same as include/pygbe.h, stated independently):
 *   panels are numbered globally, surface after surface, in the caller's triangle order;
 *   tri[j][9] = corner coordinates p0,p1,p2 of panel j; surf[j] = its surface;
 *   unknown vector x: for surface s with N_s panels starting at global panel o_s:
 *        x[2*o_s + j] = phi_j,  x[2*o_s + N_s + j] = dphi/dn_j (region_in side, normal in->out)
 *   row vector y:  y[2*o_s + j]       = equation of region_in(s)  collocated on panel j of s
 *                  y[2*o_s + N_s + j] = equation of region_out(s) collocated on panel j of s
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_OK 0
#define ORC_EINVAL (-1)

static const double ORC_PI = 3.14159265358979323846;

/* ------------------------------------------------------------------------------------------------
 * Gauss quadrature rules on the triangle, barycentric, weights summing to 1.
 * PAPER.md:163 ("Gauss quadrature"), :203 (K), :235 and Tables 4, 6 (K_fine = 19).  The paper does not
 * print the rules: K = 1, 3, 4, 7 are the classical centroid / degree-2 / degree-3 / Radon degree-5
 * rules (reading A5); K = 19 is the degree-9 S3-symmetric rule of reading A7b.
 * ---------------------------------------------------------------------------------------------- */
static int put_orbit3(double *b, double *w, int at, double a, double wt)
{   /* orbit (a, bb, bb) with bb = (1-a)/2 : 3 points */
    double bb = 0.5 * (1.0 - a);
    double p[3][3] = {{a, bb, bb}, {bb, a, bb}, {bb, bb, a}};
    for (int k = 0; k < 3; k++) { memcpy(b + 3 * (at + k), p[k], 3 * sizeof(double)); w[at + k] = wt; }
    return at + 3;
}
static int put_orbit6(double *b, double *w, int at, double a, double bb, double c, double wt)
{
    double p[6][3] = {{a, bb, c}, {a, c, bb}, {bb, a, c}, {bb, c, a}, {c, a, bb}, {c, bb, a}};
    for (int k = 0; k < 6; k++) { memcpy(b + 3 * (at + k), p[k], 3 * sizeof(double)); w[at + k] = wt; }
    return at + 6;
}

int orc_quadrature(int K, double *bary, double *w)
{
    const double third = 1.0 / 3.0;
    int at = 0;
    switch (K) {
    case 1:
        bary[0] = bary[1] = bary[2] = third; w[0] = 1.0; return ORC_OK;
    case 3:
        put_orbit3(bary, w, 0, 2.0 / 3.0, third); return ORC_OK;
    case 4:
        bary[0] = bary[1] = bary[2] = third; w[0] = -27.0 / 48.0;
        put_orbit3(bary, w, 1, 0.6, 25.0 / 48.0); return ORC_OK;
    case 7: {
        double s15 = sqrt(15.0);
        bary[0] = bary[1] = bary[2] = third; w[0] = 9.0 / 40.0;
        double b1 = (6.0 - s15) / 21.0, b2 = (6.0 + s15) / 21.0;
        at = put_orbit3(bary, w, 1, 1.0 - 2.0 * b1, (155.0 - s15) / 1200.0);
        put_orbit3(bary, w, at, 1.0 - 2.0 * b2, (155.0 + s15) / 1200.0);
        return ORC_OK; }
    case 19:
        bary[0] = bary[1] = bary[2] = third; w[0] = 0.0971357962827988;
        at = 1;
        at = put_orbit3(bary, w, at, 0.9105409732110946, 0.0255776756586980);
        at = put_orbit3(bary, w, at, 0.0206349616025247, 0.0313347002271391);
        at = put_orbit3(bary, w, at, 0.1258208170141267, 0.0778275410047743);
        at = put_orbit3(bary, w, at, 0.6235929287619345, 0.0796477389272102);
        put_orbit6(bary, w, at, 0.2219629891607657, 0.0368384120547363, 0.7411985987844980,
                   0.0432835393772894);
        return ORC_OK;
    default:
        return ORC_EINVAL;
    }
}

/* N-point Gauss-Legendre nodes and weights on [-1,1] (used by the semi-analytic self integral,
 * PAPER.md:165, :235 "N_k the number of Gauss points per side").  Newton on P_N. */
int orc_gauss_legendre(int N, double *x, double *w)
{
    if (N < 1) return ORC_EINVAL;
    for (int i = 0; i < N; i++) {
        double z = cos(ORC_PI * (i + 0.75) / (N + 0.5)), pp = 1.0;
        for (int it = 0; it < 100; it++) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 1; j <= N; j++) {
                double p3 = p2; p2 = p1;
                p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j;
            }
            pp = N * (z * p1 - p2) / (z * z - 1.0);
            double dz = p1 / pp;
            z -= dz;
            if (fabs(dz) < 1e-16) break;
        }
        x[i] = z;
        w[i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------------
 * Step 1, geometry.  PAPER.md:96 ("flat triangular panels"), :104 ("r_i corresponds to the center of
 * panel").  c = (p0+p1+p2)/3, A = |(p1-p0)x(p2-p0)|/2, n = (p1-p0)x(p2-p0)/(2A).
 * ---------------------------------------------------------------------------------------------- */
static void panel_geom(const double *t, double *c, double *n, double *A)
{
    double u[3], v[3], cr[3];
    for (int k = 0; k < 3; k++) {
        u[k] = t[3 + k] - t[k];
        v[k] = t[6 + k] - t[k];
        c[k] = (t[k] + t[3 + k] + t[6 + k]) / 3.0;
    }
    cr[0] = u[1] * v[2] - u[2] * v[1];
    cr[1] = u[2] * v[0] - u[0] * v[2];
    cr[2] = u[0] * v[1] - u[1] * v[0];
    double len = sqrt(cr[0] * cr[0] + cr[1] * cr[1] + cr[2] * cr[2]);
    *A = 0.5 * len;
    for (int k = 0; k < 3; k++) n[k] = cr[k] / len;
}

int orc_panel_geometry(long npan, const double *tri, double *centroid, double *normal, double *area)
{
    for (long j = 0; j < npan; j++) panel_geom(tri + 9 * j, centroid + 3 * j, normal + 3 * j, area + j);
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------------
 * Step 2, kernels.  PAPER.md:55-58 (eq. 2, Green's functions), :98 (eq. 9).
 *   G = exp(-kappa r)/(4 pi r),   dG/dn_y = (n.d)(1+kappa r) exp(-kappa r)/(4 pi r^3),  d = x - y,
 * n the normal at the source point y (reading A3).  kappa = 0 gives the Laplace kernel.
 * ---------------------------------------------------------------------------------------------- */
static void green(const double *x, const double *y, const double *n, double kappa, double *G, double *dG)
{
    double d0 = x[0] - y[0], d1 = x[1] - y[1], d2 = x[2] - y[2];
    double r = sqrt(d0 * d0 + d1 * d1 + d2 * d2);
    double e = exp(-kappa * r);
    *G = e / (4.0 * ORC_PI * r);
    *dG = (n[0] * d0 + n[1] * d1 + n[2] * d2) * (1.0 + kappa * r) * e / (4.0 * ORC_PI * r * r * r);
}

/* Step 3, regular entry.  PAPER.md:163: V_ij = A_j sum_g w_g G(x_i,y_jg), K_ij likewise with dG/dn. */
static void panel_quadrature(const double *x, const double *t, const double *n, double A, double kappa,
                             int K, const double *bary, const double *w, double *V, double *Kd)
{
    double sv = 0.0, sk = 0.0;
    for (int g = 0; g < K; g++) {
        double y[3], G, dG;
        for (int k = 0; k < 3; k++)
            y[k] = bary[3 * g] * t[k] + bary[3 * g + 1] * t[3 + k] + bary[3 * g + 2] * t[6 + k];
        green(x, y, n, kappa, &G, &dG);
        sv += w[g] * G;
        sk += w[g] * dG;
    }
    *V = A * sv;
    *Kd = A * sk;
}

/* Step 5, self entry (semi-analytical, "semi-analytical technique presented by Zhu et
 * al.", :235 "N_k Gauss points per side"; reading A6).  Polar coordinates about the centroid c in the
 * panel plane: for each side, h = distance from c to the side's line, theta measured from the foot of
 * the perpendicular, R(theta) = h / cos(theta); radial integral analytic:
 *     int_0^R (e^{-kappa r}/r) r dr = R (Laplace) or (1 - e^{-kappa R})/kappa (Yukawa);
 * angular integral by N_k-point Gauss-Legendre on [theta_1, theta_2].  Result carries 1/(4 pi). */
static double self_single_layer(const double *t, double kappa, int Nk, const double *glx, const double *glw)
{
    double c[3], nn[3], A;
    panel_geom(t, c, nn, &A);
    double total = 0.0;
    for (int s = 0; s < 3; s++) {
        const double *a = t + 3 * s, *b = t + 3 * ((s + 1) % 3);
        double e[3], len = 0.0;
        for (int k = 0; k < 3; k++) { e[k] = b[k] - a[k]; len += e[k] * e[k]; }
        len = sqrt(len);
        for (int k = 0; k < 3; k++) e[k] /= len;
        /* signed abscissae of a and b along the side, measured from the foot of the perpendicular */
        double sa = 0.0, sb = 0.0;
        for (int k = 0; k < 3; k++) { sa += (a[k] - c[k]) * e[k]; sb += (b[k] - c[k]) * e[k]; }
        double h2 = 0.0;
        for (int k = 0; k < 3; k++) { double p = (a[k] - c[k]) - sa * e[k]; h2 += p * p; }
        double h = sqrt(h2);
        double th1 = atan2(sa, h), th2 = atan2(sb, h);
        double half = 0.5 * (th2 - th1), mid = 0.5 * (th2 + th1), acc = 0.0;
        for (int q = 0; q < Nk; q++) {
            double th = mid + half * glx[q];
            double R = h / cos(th);
            double f = (kappa == 0.0) ? R : (1.0 - exp(-kappa * R)) / kappa;
            acc += glw[q] * f;
        }
        total += half * acc;
    }
    return total / (4.0 * ORC_PI);
}

int orc_self_entry(const double *tri9, double kappa, int Nk, double *V)
{
    if (Nk < 1 || Nk > 256) return ORC_EINVAL;
    double glx[256], glw[256];
    orc_gauss_legendre(Nk, glx, glw);
    *V = self_single_layer(tri9, kappa, Nk, glx, glw);
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------------
 * Problem description handed in by the caller (flat arrays, see header comment).
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
    long npan; const double *tri; const int *surf;
    int nsurf; const int *rin; const int *rout;
    int nreg; const double *eps; const double *kappa;
    int K, Kfine, Nk; double thres;
    /* derived */
    double *c, *n, *A; long *first; long *count;
    double bK[3 * 19], wK[19], bF[3 * 19], wF[19], glx[256], glw[256];
} orc_prob;

static int prob_init(orc_prob *P)
{
    if (P->npan <= 0 || P->nsurf <= 0 || P->nreg <= 0) return ORC_EINVAL;
    if (orc_quadrature(P->K, P->bK, P->wK) != ORC_OK) return ORC_EINVAL;
    if (orc_quadrature(P->Kfine, P->bF, P->wF) != ORC_OK) return ORC_EINVAL;
    if (P->Nk < 1 || P->Nk > 256) return ORC_EINVAL;
    orc_gauss_legendre(P->Nk, P->glx, P->glw);
    P->c = malloc(sizeof(double) * 3 * P->npan);
    P->n = malloc(sizeof(double) * 3 * P->npan);
    P->A = malloc(sizeof(double) * P->npan);
    P->first = calloc(P->nsurf, sizeof(long));
    P->count = calloc(P->nsurf, sizeof(long));
    orc_panel_geometry(P->npan, P->tri, P->c, P->n, P->A);
    /* panels of one surface must be contiguous and surfaces in increasing order */
    for (long j = 0; j < P->npan; j++) {
        int s = P->surf[j];
        if (s < 0 || s >= P->nsurf) return ORC_EINVAL;
        if (j > 0 && s < P->surf[j - 1]) return ORC_EINVAL;
        if (P->count[s] == 0) P->first[s] = j;
        P->count[s]++;
    }
    for (int s = 0; s < P->nsurf; s++) {
        if (P->rin[s] < 0 || P->rin[s] >= P->nreg || P->rout[s] < 0 || P->rout[s] >= P->nreg ||
            P->rin[s] == P->rout[s]) return ORC_EINVAL;
    }
    return ORC_OK;
}
static void prob_free(orc_prob *P)
{
    free(P->c); free(P->n); free(P->A); free(P->first); free(P->count);
}

/* Steps 3-5 put together: the matrix entries V_ij, K_ij of panel j seen from the collocation point of
 * panel i with the kernel of parameter kappa.
 *   i == j          : self entry, K_ii = 0 (flat panel, principal value; "limiting process")
 *   near-singular   : |x_i - c_j|^2 < thres^2 * 2 A_j  -> K_fine-point rule  (A7)
 *   otherwise       : K-point rule */
static void entry(const orc_prob *P, long i, long j, double kappa, double *V, double *Kd)
{
    const double *t = P->tri + 9 * j;
    if (i == j) {
        *V = self_single_layer(t, kappa, P->Nk, P->glx, P->glw);
        *Kd = 0.0;
        return;
    }
    const double *x = P->c + 3 * i, *cj = P->c + 3 * j;
    double d2 = 0.0;
    for (int k = 0; k < 3; k++) d2 += (x[k] - cj[k]) * (x[k] - cj[k]);
    if (d2 < P->thres * P->thres * 2.0 * P->A[j])
        panel_quadrature(x, t, P->n + 3 * j, P->A[j], kappa, P->Kfine, P->bF, P->wF, V, Kd);
    else
        panel_quadrature(x, t, P->n + 3 * j, P->A[j], kappa, P->K, P->bK, P->wK, V, Kd);
}

/* decode a row / unknown index into (surface, half, global panel) */
static int decode(const orc_prob *P, long r, int *s_out, int *half, long *pan)
{
    for (int s = 0; s < P->nsurf; s++) {
        long o = 2 * P->first[s], N = P->count[s];
        if (r >= o && r < o + 2 * N) {
            *s_out = s; *half = (r - o) >= N; *pan = P->first[s] + (r - o) % N;
            return 1;
        }
    }
    return 0;
}

/* Step 6, the operator.  Single surface: eq. (10).  Several surfaces: PAPER.md:121-133
 * refers to Altman et al.; the rule (reading A4) is Green's third identity written for each region
 * Omega with the normal taken outward from Omega plus eps_in dphi_in/dn = eps_out dphi_out/dn (eq. 1,
 * PAPER.md:43).  For every region Omega and every surface T in its boundary, one block row:
 *   1/2 phi_T(x_i) - sum_{S in dOmega} sigma_S [ c_S (V^Omega_TS dphi_S)_i - (K^Omega_TS phi_S)_i ]
 * sigma_S = +1, c_S = 1 if Omega = region_in(S); sigma_S = -1, c_S = eps_in(S)/eps_out(S) otherwise. */
static double operator_row(const orc_prob *P, long r, const double *x)
{
    int T, half; long i;
    if (!decode(P, r, &T, &half, &i)) return NAN;
    int Om = half ? P->rout[T] : P->rin[T];
    double kap = P->kappa[Om];
    double acc = 0.5 * x[2 * P->first[T] + (i - P->first[T])];
    for (int S = 0; S < P->nsurf; S++) {
        double sigma, c;
        if (P->rin[S] == Om) { sigma = 1.0; c = 1.0; }
        else if (P->rout[S] == Om) { sigma = -1.0; c = P->eps[P->rin[S]] / P->eps[P->rout[S]]; }
        else continue;
        const double *phi = x + 2 * P->first[S], *dphi = phi + P->count[S];
        double sv = 0.0, sk = 0.0;
        for (long jj = 0; jj < P->count[S]; jj++) {
            double V, Kd;
            entry(P, i, P->first[S] + jj, kap, &V, &Kd);
            sv += V * dphi[jj];
            sk += Kd * phi[jj];
        }
        acc -= sigma * (c * sv - sk);
    }
    return acc;
}

#define ORC_PROB_ARGS long npan, const double *tri, const int *surf, int nsurf, const int *rin,        \
                      const int *rout, int nreg, const double *eps, const double *kappa, int K,        \
                      int Kfine, double thres, int Nk
#define ORC_PROB_FILL(P) orc_prob P; memset(&P, 0, sizeof(P)); P.npan = npan; P.tri = tri; P.surf = surf; \
    P.nsurf = nsurf; P.rin = rin; P.rout = rout; P.nreg = nreg; P.eps = eps; P.kappa = kappa; P.K = K;   \
    P.Kfine = Kfine; P.thres = thres; P.Nk = Nk;                                                         \
    { int rc_ = prob_init(&P); if (rc_ != ORC_OK) { prob_free(&P); return rc_; } }

/* y[rows] = (A x)[rows].  rows == NULL: all 2*npan rows, y has 2*npan entries; otherwise y has nrows. */
int orc_matvec(ORC_PROB_ARGS, const double *x, const long *rows, long nrows, double *y)
{
    ORC_PROB_FILL(P);
    long n = rows ? nrows : 2 * npan;
#pragma omp parallel for schedule(dynamic, 8)
    for (long q = 0; q < n; q++) y[q] = operator_row(&P, rows ? rows[q] : q, x);
    prob_free(&P);
    return ORC_OK;
}

/* One matrix entry pair (V_ij, K_ij) under the kernel of `region`, for brute-force tests. */
int orc_entry(ORC_PROB_ARGS, int region, long i, long j, double *V, double *Kd)
{
    ORC_PROB_FILL(P);
    if (region < 0 || region >= nreg || i < 0 || j < 0 || i >= npan || j >= npan) { prob_free(&P); return ORC_EINVAL; }
    entry(&P, i, j, kappa[region], V, Kd);
    prob_free(&P);
    return ORC_OK;
}

/* Right-hand side, eq. (9)/(11), PAPER.md:98, :116 with the 1/(4 pi) of eq. (9) (reading A2):
 *   b[row(Omega,T,i)] = sum_{k in Omega} q_k G_Omega(x_i, r_k) / eps_Omega. */
int orc_rhs(ORC_PROB_ARGS, long nq, const double *qxyz, const double *q, const int *qreg, double *b)
{
    ORC_PROB_FILL(P);
#pragma omp parallel for schedule(static)
    for (long r = 0; r < 2 * npan; r++) {
        int T, half; long i;
        decode(&P, r, &T, &half, &i);
        int Om = half ? rout[T] : rin[T];
        double acc = 0.0;
        for (long k = 0; k < nq; k++) {
            if (qreg[k] != Om) continue;
            double d2 = 0.0;
            for (int a = 0; a < 3; a++) { double d = P.c[3 * i + a] - qxyz[3 * k + a]; d2 += d * d; }
            double rr = sqrt(d2);
            acc += q[k] * exp(-kappa[Om] * rr) / (4.0 * ORC_PI * rr);
        }
        b[r] = acc / eps[Om];
    }
    prob_free(&P);
    return ORC_OK;
}

/* Unit constant (reading A17): C0 = qe^2 N_A 1e-3 1e10 / eps0  [kJ Angstrom / (mol e^2)], chosen so
 * that the paper's analytic sphere value -41.2465 kJ/mol is reproduced. */
double orc_C0(void)
{
    const double qe = 1.60217646e-19, NA = 6.0221415e23, eps0 = 8.854187818e-12;
    return qe * qe * NA * 1e-3 * 1e10 / eps0;
}

/* Reaction potential at the charges, eq. (4) PAPER.md:68 (discretised, :119), generalised to the
 * boundary of the charge's region with the sigma / c rule of operator_row; plain K-point quadrature.
 * phi_reac[k] for every charge; then eq. (6): dG_solv = 1/2 C0 sum_k q_k phi_reac(r_k). */
int orc_reaction_potential(ORC_PROB_ARGS, long nq, const double *qxyz, const int *qreg, const double *x,
                           double *phi_reac)
{
    ORC_PROB_FILL(P);
#pragma omp parallel for schedule(dynamic, 1)
    for (long k = 0; k < nq; k++) {
        int Om = qreg[k];
        double acc = 0.0;
        for (int S = 0; S < nsurf; S++) {
            double sigma, c;
            if (rin[S] == Om) { sigma = 1.0; c = 1.0; }
            else if (rout[S] == Om) { sigma = -1.0; c = eps[rin[S]] / eps[rout[S]]; }
            else continue;
            const double *phi = x + 2 * P.first[S], *dphi = phi + P.count[S];
            double sv = 0.0, sk = 0.0;
            for (long jj = 0; jj < P.count[S]; jj++) {
                long j = P.first[S] + jj;
                double V, Kd;
                panel_quadrature(qxyz + 3 * k, tri + 9 * j, P.n + 3 * j, P.A[j], kappa[Om], K, P.bK, P.wK, &V, &Kd);
                sv += V * dphi[jj];
                sk += Kd * phi[jj];
            }
            acc += sigma * (c * sv - sk);
        }
        phi_reac[k] = acc;
    }
    prob_free(&P);
    return ORC_OK;
}

int orc_solvation_energy(long nq, const double *q, const double *phi_reac, double *E_kJ_mol)
{
    double s = 0.0;
    for (long k = 0; k < nq; k++) s += q[k] * phi_reac[k];
    *E_kJ_mol = 0.5 * orc_C0() * s;
    return ORC_OK;
}

/* Coulomb energy of the point charges, eq. (8) PAPER.md:87-90:
 *   dG_Coul = 1/2 C0 sum_{k != l, same region} q_k q_l / (4 pi eps_Omega r_kl). */
int orc_coulomb_energy(long nq, const double *qxyz, const double *q, const int *qreg, int nreg,
                       const double *eps, double *E_kJ_mol)
{
    double s = 0.0;
    for (long k = 0; k < nq; k++)
        for (long l = 0; l < nq; l++) {
            if (k == l || qreg[k] != qreg[l]) continue;
            if (qreg[k] < 0 || qreg[k] >= nreg) return ORC_EINVAL;
            double d2 = 0.0;
            for (int a = 0; a < 3; a++) { double d = qxyz[3 * k + a] - qxyz[3 * l + a]; d2 += d * d; }
            s += q[k] * q[l] / (4.0 * ORC_PI * eps[qreg[k]] * sqrt(d2));
        }
    *E_kJ_mol = 0.5 * orc_C0() * s;
    return ORC_OK;
}

/* Double-layer potential of a unit density (and single-layer) at an arbitrary point, K-point rule,
 * no near-field treatment: used by the Gauss-identity test at interior / exterior points. */
int orc_layer_potentials_at(ORC_PROB_ARGS, int region, long npts, const double *pts, double *V, double *Kd)
{
    ORC_PROB_FILL(P);
    for (long p = 0; p < npts; p++) {
        double sv = 0.0, sk = 0.0;
        for (long j = 0; j < npan; j++) {
            double v, k;
            panel_quadrature(pts + 3 * p, tri + 9 * j, P.n + 3 * j, P.A[j], kappa[region], K, P.bK, P.wK, &v, &k);
            sv += v; sk += k;
        }
        V[p] = sv; Kd[p] = sk;
    }
    prob_free(&P);
    return ORC_OK;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
