// tables.cuh -- quadrature rules (host side, handed to kernels by value) and the multi-index tables of
// the Cartesian Taylor expansion (one device-memory copy per handle, valid for every P <= PYGBE_PMAX).
#pragma once
#include "common.cuh"

// Gauss rules on the triangle in barycentric coordinates, weights summing to 1 ("Gauss
// quadrature"; K in Tables 1, 3 :197-225; K_fine = 19 in Tables 4, 6 :237-278).  The paper prints no
// rule; readings A5 (K = 1, 3, 4, 7) and A7b (19-point degree-9 rule).
struct QuadTables {
    int K, Kfine, Nk;
    double bK[7][3], wK[7];
    double bF[19][3], wF[19];
    double glx[64], glw[64];        // Gauss-Legendre on [-1,1] for the semi-analytic self integral
};

static void orbit3(double (*b)[3], double *w, int &at, double a, double wt)
{
    double r = 0.5 * (1.0 - a);
    for (int k = 0; k < 3; k++) {
        b[at][0] = b[at][1] = b[at][2] = r;
        b[at][k] = a;
        w[at++] = wt;
    }
}
static void orbit6(double (*b)[3], double *w, int &at, double a, double bb, double c, double wt)
{
    const double v[3] = {a, bb, c};
    const int perm[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
    for (int k = 0; k < 6; k++) {
        for (int i = 0; i < 3; i++) b[at][i] = v[perm[k][i]];
        w[at++] = wt;
    }
}

static int fill_triangle_rule(int K, double (*b)[3], double *w)
{
    int at = 0;
    const double t = 1.0 / 3.0;
    if (K == 1) {
        b[0][0] = b[0][1] = b[0][2] = t; w[0] = 1.0;
    } else if (K == 3) {
        orbit3(b, w, at, 2.0 / 3.0, t);
    } else if (K == 4) {
        b[0][0] = b[0][1] = b[0][2] = t; w[0] = -27.0 / 48.0; at = 1;
        orbit3(b, w, at, 0.6, 25.0 / 48.0);
    } else if (K == 7) {
        const double s = std::sqrt(15.0);
        b[0][0] = b[0][1] = b[0][2] = t; w[0] = 9.0 / 40.0; at = 1;
        orbit3(b, w, at, 1.0 - 2.0 * (6.0 - s) / 21.0, (155.0 - s) / 1200.0);
        orbit3(b, w, at, 1.0 - 2.0 * (6.0 + s) / 21.0, (155.0 + s) / 1200.0);
    } else if (K == 19) {
        b[0][0] = b[0][1] = b[0][2] = t; w[0] = 0.0971357962827988; at = 1;
        orbit3(b, w, at, 0.9105409732110946, 0.0255776756586980);
        orbit3(b, w, at, 0.0206349616025247, 0.0313347002271391);
        orbit3(b, w, at, 0.1258208170141267, 0.0778275410047743);
        orbit3(b, w, at, 0.6235929287619345, 0.0796477389272102);
        orbit6(b, w, at, 0.2219629891607657, 0.0368384120547363, 0.7411985987844980, 0.0432835393772894);
    } else {
        return PYGBE_EINVAL;
    }
    return PYGBE_OK;
}

static void fill_gauss_legendre(int N, double *x, double *w)
{
    // roots of P_N by Newton from the Chebyshev guess; standard three-term recurrence
    const double pi = 3.14159265358979323846;
    for (int i = 0; i < N; i++) {
        double z = std::cos(pi * (i + 0.75) / (N + 0.5)), dp = 1.0;
        for (int it = 0; it < 100; it++) {
            double p0 = 1.0, p1 = z;
            for (int k = 2; k <= N; k++) {
                double p2 = ((2.0 * k - 1.0) * z * p1 - (k - 1.0) * p0) / k;
                p0 = p1; p1 = p2;
            }
            if (N == 1) { p0 = 1.0; p1 = z; }
            dp = N * (z * p1 - p0) / (z * z - 1.0);
            double dz = p1 / dp;
            z -= dz;
            if (std::fabs(dz) < 1e-16) break;
        }
        x[i] = z;
        w[i] = 2.0 / ((1.0 - z * z) * dp * dp);
    }
}

static int make_quad_tables(int K, int Kfine, int Nk, QuadTables *q)
{
    memset(q, 0, sizeof(*q));
    if (!(K == 1 || K == 3 || K == 4 || K == 7)) {
        pygbe_set_error("K = %d: supported Gauss rules are 1, 3, 4, 7", K);
        return PYGBE_EINVAL;
    }
    if (!(Kfine == 1 || Kfine == 3 || Kfine == 4 || Kfine == 7 || Kfine == 19)) {
        pygbe_set_error("K_fine = %d: supported rules are 1, 3, 4, 7, 19", Kfine);
        return PYGBE_EINVAL;
    }
    if (Nk < 1 || Nk > 64) {
        pygbe_set_error("N_k = %d out of range 1..64", Nk);
        return PYGBE_EINVAL;
    }
    q->K = K; q->Kfine = Kfine; q->Nk = Nk;
    fill_triangle_rule(K, q->bK, q->wK);
    fill_triangle_rule(Kfine, q->bF, q->wF);
    fill_gauss_legendre(Nk, q->glx, q->glw);
    return PYGBE_OK;
}

// ---------------------------------------------------------------------------------------------------
// Multi-index tables.  Canonical order of the coefficients k = (kx,ky,kz), |k| <= P: by total order n,
// then kx descending, then ky descending.  The first Nc(P') entries are the set for any P' <= PMAX.
// One copy lives in device memory per handle; kernels stage what they need into shared memory.
struct IndexTables {
    unsigned char kxyz[PYGBE_NCMAX][4];                              // kx, ky, kz, n
    short idx3[PYGBE_PMAX + 1][PYGBE_PMAX + 1][PYGBE_PMAX + 1];       // -> canonical index (or -1)
    double binom[PYGBE_PMAX + 1][PYGBE_PMAX + 1];
};

static void fill_index_tables(IndexTables *t)
{
    memset(t->idx3, 0xff, sizeof(t->idx3));
    int at = 0;
    for (int n = 0; n <= PYGBE_PMAX; n++)
        for (int kx = n; kx >= 0; kx--)
            for (int ky = n - kx; ky >= 0; ky--) {
                int kz = n - kx - ky;
                t->kxyz[at][0] = kx; t->kxyz[at][1] = ky; t->kxyz[at][2] = kz; t->kxyz[at][3] = n;
                t->idx3[kx][ky][kz] = (short)at++;
            }
    for (int n = 0; n <= PYGBE_PMAX; n++)
        for (int m = 0; m <= PYGBE_PMAX; m++) {
            if (m > n) { t->binom[n][m] = 0; continue; }
            t->binom[n][m] = (m == 0 || m == n) ? 1.0 : t->binom[n - 1][m - 1] + t->binom[n - 1][m];
        }
}

// The regrouping of the Taylor series used by the M2P (m2p.cuh), on HARMONICALLY REDUCED moments.
//
// G = exp(-kappa r) / r satisfies (laplace_y - kappa^2) G = 0 away from the source, so its Taylor coefficients
// a^k = (1/k!) D_y^k G obey
//     (kx+1)(kx+2) a^(k+2ex) + (ky+1)(ky+2) a^(k+2ey) + (kz+1)(kz+2) a^(k+2ez) = kappa^2 a^k
// and every a^k with kz >= 2 is a combination of coefficients with smaller kz of the same and of lower order (all
// within |k| <= P).  Moving the moments accordingly, from kz = P down to 2,
//     Mt^k        += kappa^2 / ((kz+1)(kz+2)) M^(k+2ez)
//     Mt^(k+2ex)  -= (kx+1)(kx+2) / ((kz+1)(kz+2)) M^(k+2ez),      Mt^(k+2ey) likewise,
// leaves the truncated series unchanged, sum_{|k|<=P} a^k M^k = sum_{|k|<=P, kz<=1} a^k Mt^k (an identity of the series,
// not an approximation: checked to 1e-16 against the unreduced form, coefficient growth <= 54 at P = 12), with only
// (P+1)^2 moments left instead of Nc -- 81 instead of 165 at P = 8.  The regrouping of m2p.cuh applied to Mt then has
// ez <= 1 and jz = 0 only: entry p of the W stream -- ex, ey ascending, ez in {0, 1}, |e| <= P, then J = 0 ..
// (P - |e|) / 2, m = |e| + J -- is
//     W_p = (-1)^|e| / e!  sum_{|j| = J, jz = 0} Mt^(e + 2j) / (2^J j!),
// 165 entries at P = 8 (295 unreduced) against 80 monomials d^e (164).  Reduction and regrouping are composed here, once
// per kappa, into a sparse row over the canonical index of the ORIGINAL moments: W_p = sum_{i in [off[p], off[p+1])}
// c[i] M^(k[i]); the P2M / M2M epilogue (farfield.cuh) applies it in fp64.
struct WTable {
    std::vector<int> off;
    std::vector<short> k;
    std::vector<double> c;
    std::vector<short> deg;          // Laplace form only: |f| of entry p (the power of the cell edge it is divided by)
};
static void build_w_table(int P, double kappa, const IndexTables &t, WTable *w)
{
    double fact[PYGBE_PMAX + 1];
    fact[0] = 1.0;
    for (int i = 1; i <= PYGBE_PMAX; i++) fact[i] = fact[i - 1] * i;
    const int Nc = (P + 1) * (P + 2) * (P + 3) / 6;
    // D: reduced moments as rows over the original ones, Mt = D M
    std::vector<double> D((size_t)Nc * Nc, 0.0), row(Nc);
    for (int i = 0; i < Nc; i++) D[(size_t)i * Nc + i] = 1.0;
    for (int Kz = P; Kz >= 2; Kz--)
        for (int K = 0; K < Nc; K++) {
            if (t.kxyz[K][2] != Kz) continue;
            const int kx = t.kxyz[K][0], ky = t.kxyz[K][1], kz = Kz - 2;
            const double den = (kz + 1.0) * (kz + 2.0);
            std::copy(D.begin() + (size_t)K * Nc, D.begin() + (size_t)(K + 1) * Nc, row.begin());
            std::fill(D.begin() + (size_t)K * Nc, D.begin() + (size_t)(K + 1) * Nc, 0.0);
            double *lo = &D[(size_t)t.idx3[kx][ky][kz] * Nc], *xx = &D[(size_t)t.idx3[kx + 2][ky][kz] * Nc], *yy = &D[(size_t)t.idx3[kx][ky + 2][kz] * Nc];
            const double cl = kappa * kappa / den, cx = (kx + 1.0) * (kx + 2.0) / den, cy = (ky + 1.0) * (ky + 2.0) / den;
            for (int i = 0; i < Nc; i++) { lo[i] += cl * row[i]; xx[i] -= cx * row[i]; yy[i] -= cy * row[i]; }
        }
    w->off.assign(1, 0); w->k.clear(); w->c.clear(); w->deg.clear();
    for (int ex = 0; ex <= P; ex++)
        for (int ey = 0; ey <= P - ex; ey++)
            for (int ez = 0; ez <= std::min(1, P - ex - ey); ez++) {
                const int n = ex + ey + ez;
                const double pre = ((n & 1) ? -1.0 : 1.0) / (fact[ex] * fact[ey] * fact[ez]);
                for (int J = 0; J <= (P - n) / 2; J++) {
                    std::fill(row.begin(), row.end(), 0.0);
                    for (int jx = J; jx >= 0; jx--) {
                        const int jy = J - jx;
                        const double cj = pre / (std::ldexp(1.0, J) * fact[jx] * fact[jy]);
                        const double *src = &D[(size_t)t.idx3[ex + 2 * jx][ey + 2 * jy][ez] * Nc];
                        for (int i = 0; i < Nc; i++) row[i] += cj * src[i];
                    }
                    for (int i = 0; i < Nc; i++)
                        if (row[i] != 0.0) { w->k.push_back((short)i); w->c.push_back(row[i]); }
                    w->off.push_back((int)w->k.size());
                }
            }
}

// The Laplace form of the series (m2p.cuh, k_m2p_lap): entry p of the stream -- ex, ey, ez DESCENDING with
// |f| <= P, the order the nested Horner scheme consumes them -- is the coefficient of u^f, u = d / r^2,
//     C_f = sum_{2i <= f, e = f - 2i, J = |i|} (J! / i!) sum_{|j| = J} (-1)^J (2(|e| + J) - 1)!! / (e! 2^J j!) M^(e + 2j),
// again a sparse row over the canonical moment index (1275 non-zeros at P = 8).  (-1)!! = 1.
static void build_lap_table(int P, const IndexTables &t, WTable *w)
{
    double fact[PYGBE_PMAX + 1], dfact[2 * PYGBE_PMAX + 2];
    fact[0] = 1.0;
    for (int i = 1; i <= PYGBE_PMAX; i++) fact[i] = fact[i - 1] * i;
    for (int n = 0; n <= PYGBE_PMAX; n++) {                          // dfact[n] = (2n - 1)!!
        dfact[n] = 1.0;
        for (int q = 2 * n - 1; q > 1; q -= 2) dfact[n] *= q;
    }
    w->off.assign(1, 0); w->k.clear(); w->c.clear(); w->deg.clear();
    std::vector<double> row(PYGBE_NCMAX);
    for (int fx = P; fx >= 0; fx--)
        for (int fy = P - fx; fy >= 0; fy--)
            for (int fz = P - fx - fy; fz >= 0; fz--) {
                std::fill(row.begin(), row.end(), 0.0);
                for (int ix = 0; ix <= fx / 2; ix++)
                    for (int iy = 0; iy <= fy / 2; iy++)
                        for (int iz = 0; iz <= fz / 2; iz++) {
                            const int J = ix + iy + iz, ex = fx - 2 * ix, ey = fy - 2 * iy, ez = fz - 2 * iz, ne = ex + ey + ez;
                            const double pre = ((J & 1) ? -1.0 : 1.0) * dfact[ne + J] * fact[J] /
                                               (fact[ex] * fact[ey] * fact[ez] * std::ldexp(1.0, J) * fact[ix] * fact[iy] * fact[iz]);
                            for (int jx = J; jx >= 0; jx--)
                                for (int jy = J - jx; jy >= 0; jy--) {
                                    const int jz = J - jx - jy;
                                    row[t.idx3[ex + 2 * jx][ey + 2 * jy][ez + 2 * jz]] += pre / (fact[jx] * fact[jy] * fact[jz]);
                                }
                        }
                for (int k = 0; k < PYGBE_NCMAX; k++)
                    if (row[k] != 0.0) { w->k.push_back((short)k); w->c.push_back(row[k]); }
                w->off.push_back((int)w->k.size());
                w->deg.push_back((short)(fx + fy + fz));
            }
}
