/*
 * lya_oracle.c -- CPU ORACLE for the Lya2pcf pixel-pair hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct C that follows the
 * paper's definitions literally.  It shares no code with the CUDA path
 * (paper_2507_00129_b200/csrc) and neither side includes or links the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call it.
 *
 * What it computes (citations are /root/reference/PAPER.md line : equation):
 *   orc_xi     -- eq. 2.4: for every listed pair of DIFFERENT
 *                 forests and every pixel pair (i,j): if the separation
 *                 (r_par, r_perp) lies inside the grid, add w_i d_i w_j d_j to
 *                 S[A], w_i w_j to W[A], 1 to N[A].  xi[A] = S[A]/W[A].
 *   orc_eta    -- eq. 2.7: the explicit n x n matrix eta.
 *   orc_dmat   -- eq. 2.6: the naive quadruple sum with the
 *                 explicit eta matrices; no use of the rank-2 structure.
 *   orc_dmat_collapsed -- CROSS-CHECK ONLY (pin PD4): the same D evaluated via
 *                 the identity-minus-rank-2 form of eta; never the definition.
 *   orc_keep   -- the seeded pixel-pair keep mask (an integer
 *                 function shared by SPECIFICATION with the CUDA path).
 *   orc_pairs_* -- forest-pair lists by brute force over all p<q (with the
 *                 oracle's own conservative |du_z| pre-filter for big N).
 *
 * Readings where the paper is silent:
 *   geometry G2-G6: s = 0.5*sqrt(|u_p-u_q|^2) = sin(theta/2), c = sqrt(1-s*s),
 *   r_par = |chi_i-chi_j|*c, r_perp = (chi_i+chi_j)*s, in-grid iff r_par <
 *   rpar_max and r_perp < rperp_max, b = (int)(r*(n/r_max)) clamped to n-1,
 *   A = n_perp*b_par + b_perp.  Every operation is one separately rounded
 *   IEEE binary64 operation (build with -ffp-contract=off, no fast-math).
 *
 * Pins: tests/test_oracle_pins.py (P1-P8, PD1-PD8 of DESIGN.md).
 * Parity unpinned: that the (r_par, r_perp) convention and the bin flattening
 * equal the authors' code -- the paper prints neither formula nor example.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int64_t n_forest, n_pix;
    const double *ux, *uy, *uz;   /* [n_forest] unit vectors (inputs, reading G1) */
    const int64_t *pix_off;       /* [n_forest+1] */
    const double *chi, *w, *delta, *loglam; /* [n_pix] */
} orc_forests;

typedef struct { double rpar_max, rperp_max; int32_t n_par, n_perp; } orc_binning;

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- geometry, operation by operation (readings G2-G6) ------------------- */

/* G2-G3: s = sin(theta/2), c = cos(theta/2) of a forest pair from the chord. */
void orc_pair_sc(const orc_forests *f, int64_t p, int64_t q, double *s, double *c)
{
    double dx = f->ux[p] - f->ux[q];
    double dy = f->uy[p] - f->uy[q];
    double dz = f->uz[p] - f->uz[q];
    double h2 = ((dx * dx) + (dy * dy)) + (dz * dz);
    *s = 0.5 * sqrt(h2);
    *c = sqrt(1.0 - ((*s) * (*s)));
}

/* G4: listed iff (chi_min_p + chi_min_q) * s < rperp_max, chi_min = first pixel. */
static int pair_listed(const orc_forests *f, const orc_binning *b, int64_t p, int64_t q)
{
    if (f->pix_off[p + 1] == f->pix_off[p] || f->pix_off[q + 1] == f->pix_off[q]) return 0;
    double s, c;
    orc_pair_sc(f, p, q, &s, &c);
    double t = f->chi[f->pix_off[p]] + f->chi[f->pix_off[q]];
    return (t * s) < b->rperp_max;
}

/* G5-G6: bin of one pixel pair; returns -1 when outside the grid. */
static inline int32_t pix_bin(const orc_binning *b, double s, double c, double chi_i, double chi_j)
{
    double d = chi_i - chi_j;
    double rpar = fabs(d) * c;
    double t = chi_i + chi_j;
    double rperp = t * s;
    if (!(rpar < b->rpar_max) || !(rperp < b->rperp_max)) return -1;
    double inv_par = (double)b->n_par / b->rpar_max;
    double inv_perp = (double)b->n_perp / b->rperp_max;
    int32_t bpar = (int32_t)(rpar * inv_par);
    int32_t bperp = (int32_t)(rperp * inv_perp);
    if (bpar >= b->n_par) bpar = b->n_par - 1;
    if (bperp >= b->n_perp) bperp = b->n_perp - 1;
    return b->n_perp * bpar + bperp;
}

/* exported for the hand-built pins (P6) */
int32_t orc_pix_bin(const orc_binning *b, double s, double c, double chi_i, double chi_j)
{
    return pix_bin(b, s, c, chi_i, chi_j);
}

/* ---- forest-pair lists ---------------------------------------------------- */

/* All p<q over the whole catalogue with NO criterion (configs[0] brute force). */
int64_t orc_pairs_all(int64_t n_forest, int32_t *pq)
{
    int64_t k = 0;
    for (int64_t p = 0; p < n_forest; ++p)
        for (int64_t q = p + 1; q < n_forest; ++q) {
            if (pq) { pq[2 * k] = (int32_t)p; pq[2 * k + 1] = (int32_t)q; }
            ++k;
        }
    return k;
}

/* Brute-force neighbour list: every p<q tested with criterion G4.  Call with
 * pq == NULL to count.  Output order: p ascending, q ascending. */
int64_t orc_pairs_brute(const orc_forests *f, const orc_binning *b, int32_t *pq)
{
    int64_t k = 0;
    for (int64_t p = 0; p < f->n_forest; ++p)
        for (int64_t q = p + 1; q < f->n_forest; ++q)
            if (pair_listed(f, b, p, q)) {
                if (pq) { pq[2 * k] = (int32_t)p; pq[2 * k + 1] = (int32_t)q; }
                ++k;
            }
    return k;
}

/* Same set as orc_pairs_brute for big N: the oracle's OWN conservative
 * pre-filter.  |u_z,p - u_z,q| <= chord = 2 s, and a listed pair has
 * s < rperp_max / (2 chi_min_global), so only forests within that u_z window
 * (found in a u_z-sorted order) are tested with G4.  Checked against
 * orc_pairs_brute in the pins (P1).  Output order: p ascending, q ascending. */
typedef struct { double uz; int64_t id; } uz_rec;
static int uz_cmp(const void *a, const void *b)
{
    double x = ((const uz_rec *)a)->uz, y = ((const uz_rec *)b)->uz;
    return (x > y) - (x < y);
}
static int i32_cmp(const void *a, const void *b)
{
    int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
    return (x > y) - (x < y);
}
int64_t orc_pairs_window(const orc_forests *f, const orc_binning *b, int32_t *pq, int64_t cap)
{
    int64_t n = f->n_forest;
    if (n < 2) return 0;
    double chi_min = INFINITY;
    for (int64_t p = 0; p < n; ++p)
        if (f->pix_off[p + 1] > f->pix_off[p] && f->chi[f->pix_off[p]] < chi_min)
            chi_min = f->chi[f->pix_off[p]];
    double smax = b->rperp_max / (2.0 * chi_min);
    double win = (smax >= 1.0 ? 2.0 : 2.0 * smax) * (1.0 + 1e-9) + 1e-12;
    uz_rec *r = (uz_rec *)malloc(sizeof(uz_rec) * (size_t)n);
    int64_t *pos = (int64_t *)malloc(sizeof(int64_t) * (size_t)n);
    for (int64_t p = 0; p < n; ++p) { r[p].uz = f->uz[p]; r[p].id = p; }
    qsort(r, (size_t)n, sizeof(uz_rec), uz_cmp);
    for (int64_t k = 0; k < n; ++k) pos[r[k].id] = k;
    int64_t total = 0;
    int32_t *tmp = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);
    for (int64_t p = 0; p < n; ++p) {
        int64_t m = 0, k0 = pos[p];
        for (int64_t k = k0 - 1; k >= 0 && f->uz[p] - r[k].uz <= win; --k)
            if (r[k].id > p && pair_listed(f, b, p, r[k].id)) tmp[m++] = (int32_t)r[k].id;
        for (int64_t k = k0 + 1; k < n && r[k].uz - f->uz[p] <= win; ++k)
            if (r[k].id > p && pair_listed(f, b, p, r[k].id)) tmp[m++] = (int32_t)r[k].id;
        qsort(tmp, (size_t)m, sizeof(int32_t), i32_cmp);
        if (pq) {
            if (total + m > cap) { total = -1; break; }
            for (int64_t t = 0; t < m; ++t) { pq[2 * (total + t)] = (int32_t)p; pq[2 * (total + t) + 1] = tmp[t]; }
        }
        total += m;
    }
    free(tmp); free(pos); free(r);
    return total;
}

/* ---- O-xi: eq. 2.4, naive double loop over pixel pairs --------------------- */
/*
 * Outputs (all [n_par*n_perp] unless noted), zeroed here:
 *   S    = sum (w_i d_i)(w_j d_j)       W = sum w_i w_j       N = pair count
 *   xi   = S/W (0 where W == 0, reading R-6)
 *   Sabs = sum |term of S|  Q = sum (w_i w_j)^2   (tolerance floors / pin P5)
 *   n_out[0] = pixel pairs of listed forest pairs that fall outside the grid
 * Accumulators are long double so the oracle is the more accurate side.
 */
void orc_xi(const orc_forests *f, const orc_binning *b, const int32_t *pq, int64_t n_pairs,
            double *S, double *W, uint64_t *N, double *xi, double *Sabs, double *Q,
            uint64_t *n_out)
{
    int32_t nb = b->n_par * b->n_perp;
    long double *gS = (long double *)calloc((size_t)nb, sizeof(long double));
    long double *gW = (long double *)calloc((size_t)nb, sizeof(long double));
    long double *gA = (long double *)calloc((size_t)nb, sizeof(long double));
    long double *gQ = (long double *)calloc((size_t)nb, sizeof(long double));
    memset(N, 0, sizeof(uint64_t) * (size_t)nb);
    uint64_t gout = 0;
#pragma omp parallel
    {
        long double *tS = (long double *)calloc((size_t)nb, sizeof(long double));
        long double *tW = (long double *)calloc((size_t)nb, sizeof(long double));
        long double *tA = (long double *)calloc((size_t)nb, sizeof(long double));
        long double *tQ = (long double *)calloc((size_t)nb, sizeof(long double));
        uint64_t *tN = (uint64_t *)calloc((size_t)nb, sizeof(uint64_t));
        uint64_t tout = 0;
#pragma omp for schedule(dynamic, 256)
        for (int64_t k = 0; k < n_pairs; ++k) {
            int64_t p = pq[2 * k], q = pq[2 * k + 1];
            double s, c;
            orc_pair_sc(f, p, q, &s, &c);
            for (int64_t i = f->pix_off[p]; i < f->pix_off[p + 1]; ++i)
                for (int64_t j = f->pix_off[q]; j < f->pix_off[q + 1]; ++j) {
                    int32_t A = pix_bin(b, s, c, f->chi[i], f->chi[j]);
                    if (A < 0) { ++tout; continue; }
                    double ww = f->w[i] * f->w[j];
                    double term = (f->w[i] * f->delta[i]) * (f->w[j] * f->delta[j]);
                    tS[A] += term;
                    tW[A] += ww;
                    tA[A] += fabs(term);
                    tQ[A] += ww * ww;
                    tN[A] += 1;
                }
        }
#pragma omp critical
        {
            for (int32_t a = 0; a < nb; ++a) {
                gS[a] += tS[a]; gW[a] += tW[a]; gA[a] += tA[a]; gQ[a] += tQ[a]; N[a] += tN[a];
            }
            gout += tout;
        }
        free(tS); free(tW); free(tA); free(tQ); free(tN);
    }
    for (int32_t a = 0; a < nb; ++a) {
        S[a] = (double)gS[a]; W[a] = (double)gW[a];
        if (Sabs) Sabs[a] = (double)gA[a];
        if (Q) Q[a] = (double)gQ[a];
        if (xi) xi[a] = (gW[a] != 0.0L) ? (double)(gS[a] / gW[a]) : 0.0;
    }
    if (n_out) n_out[0] = gout;
    free(gS); free(gW); free(gA); free(gQ);
}

/* Per-bin weighted sums of the pixel-pair coordinates (NEXT-1, second half; "mimics PICCA":
 * the correlation is tabulated with the weighted mean r_par, r_perp and redshift of the pairs of each
 * bin).  For every listed forest pair and every in-grid pixel pair (i, j), A = its bin,
 * om = w_i w_j (the weight of eq. 2.4's denominator):
 *     Rpar[A] += om * r_par,   Rperp[A] += om * r_perp,   Z[A] += om * 0.5 * (z_i + z_j),   W[A] += om
 * with r_par = |chi_i - chi_j| c and r_perp = (chi_i + chi_j) s exactly as binned (reading G5) and z the
 * caller's per-pixel redshift (reading R-19: the pair redshift is the mean of the two pixel redshifts).
 * The outputs are SUMS; the weighted means are Rpar[A] / W[A] etc. */
void orc_xi_means(const orc_forests *f, const orc_binning *b, const int32_t *pq, int64_t n_pairs, const double *z,
                  double *Rpar, double *Rperp, double *Z, double *W)
{
    int32_t nb = b->n_par * b->n_perp;
    long double *g = (long double *)calloc((size_t)nb * 4, sizeof(long double));
#pragma omp parallel
    {
        long double *t = (long double *)calloc((size_t)nb * 4, sizeof(long double));
#pragma omp for schedule(dynamic, 256)
        for (int64_t k = 0; k < n_pairs; ++k) {
            int64_t p = pq[2 * k], q = pq[2 * k + 1];
            double s, c;
            orc_pair_sc(f, p, q, &s, &c);
            for (int64_t i = f->pix_off[p]; i < f->pix_off[p + 1]; ++i)
                for (int64_t j = f->pix_off[q]; j < f->pix_off[q + 1]; ++j) {
                    int32_t A = pix_bin(b, s, c, f->chi[i], f->chi[j]);
                    if (A < 0) continue;
                    double om = f->w[i] * f->w[j];
                    double rpar = fabs(f->chi[i] - f->chi[j]) * c;
                    double rperp = (f->chi[i] + f->chi[j]) * s;
                    double zz = 0.5 * (z[i] + z[j]);
                    t[4 * A + 0] += (long double)om * rpar;
                    t[4 * A + 1] += (long double)om * rperp;
                    t[4 * A + 2] += (long double)om * zz;
                    t[4 * A + 3] += om;
                }
        }
#pragma omp critical
        for (int32_t a = 0; a < 4 * nb; ++a) g[a] += t[a];
        free(t);
    }
    for (int32_t a = 0; a < nb; ++a) {
        Rpar[a] = (double)g[4 * a]; Rperp[a] = (double)g[4 * a + 1]; Z[a] = (double)g[4 * a + 2]; W[a] = (double)g[4 * a + 3];
    }
    free(g);
}

/* ---- eq. 2.7: explicit eta for one forest (reading R-10) -------------------- */
/*
 * eta[i*n+k] = delta^K_ik - w_k/sum(w) - (L_i-Lbar) w_k (L_k-Lbar) / sum_m w_m (L_m-Lbar)^2
 * with Lbar the w-WEIGHTED mean of L = log lambda.  Returns 0, or 1 when the
 * forest is degenerate (sum w == 0 or sum w (L-Lbar)^2 == 0; reading R-7).
 */
int orc_eta(int64_t n, const double *w, const double *loglam, double *eta)
{
    long double sw = 0, swl = 0;
    for (int64_t k = 0; k < n; ++k) { sw += w[k]; swl += (long double)w[k] * loglam[k]; }
    if (!(sw > 0)) return 1;
    double lbar = (double)(swl / sw);
    long double v = 0;
    for (int64_t k = 0; k < n; ++k) { double u = loglam[k] - lbar; v += (long double)w[k] * u * u; }
    if (!(v > 0)) return 1;
    double dsw = (double)sw, dv = (double)v;
    for (int64_t i = 0; i < n; ++i)
        for (int64_t k = 0; k < n; ++k) {
            double kron = (i == k) ? 1.0 : 0.0;
            eta[i * n + k] = kron - w[k] / dsw
                           - (loglam[i] - lbar) * w[k] * (loglam[k] - lbar) / dv;
        }
    return 0;
}

/* ---- seeded pixel-pair keep mask ------------------------- */
static inline uint64_t mix64(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
uint64_t orc_mask_threshold(double reject_fraction)
{
    double t = floor(reject_fraction * 4294967296.0 + 0.5);
    if (t < 0) t = 0;
    if (t > 4294967296.0) t = 4294967296.0;
    return (uint64_t)t;
}
/* keep(seed, a, b): a, b = offsets of the two pixels in the flat arrays. */
int orc_keep(uint64_t seed, int64_t a, int64_t b, uint64_t threshold)
{
    uint64_t lo = (uint64_t)(a < b ? a : b), hi = (uint64_t)(a < b ? b : a);
    uint64_t klo = mix64(seed + lo * 0x9E3779B97F4A7C15ULL);
    uint64_t khi = mix64((seed ^ 0xD1B54A32D192ED03ULL) + hi * 0x9E3779B97F4A7C15ULL);
    uint64_t x = klo + khi;
    x ^= x >> 32;
    x *= 0xD6E8FEB86659FD93ULL;
    return (x >> 32) >= threshold;
}

/* ---- O-D: eq. 2.6, naive quadruple sum with explicit eta ------------------- */
/*
 * For every listed forest pair, every in-grid pixel pair (i,j) with
 * keep(i,j) = 1 (the mask applies to the OUTER pair only, reading R-8),
 * A = bin(i,j), om = w_i w_j:
 *     Wd[A] += om
 *     for every i' in p, j' in q:  B = bin(i',j')
 *         in-grid:  Dn[A][B]  += om * eta_p[i][i'] * eta_q[j][j']
 *         else:     Dover[A]  += (same term)         (pin PD3 only)
 * D[A][B] = Dn[A][B]/Wd[A]  (row 0 where Wd[A] == 0, reading R-6).
 * Returns 0, or 1 if some forest is degenerate (R-7).
 * Dn, D: [NB*NB] row-major [A][B]; Wd, Dover: [NB]; n_kept: [1].  D may be NULL.
 */
int orc_dmat(const orc_forests *f, const orc_binning *b, const int32_t *pq, int64_t n_pairs,
             double reject_fraction, uint64_t seed,
             double *Dn, double *Wd, double *Dover, uint64_t *n_kept, double *D)
{
    int64_t nb = (int64_t)b->n_par * b->n_perp;
    uint64_t thr = orc_mask_threshold(reject_fraction);
    memset(Dn, 0, sizeof(double) * (size_t)(nb * nb));
    memset(Wd, 0, sizeof(double) * (size_t)nb);
    if (Dover) memset(Dover, 0, sizeof(double) * (size_t)nb);
    uint64_t kept = 0;
    int bad = 0;
#pragma omp parallel
    {
        double *tD = (double *)calloc((size_t)(nb * nb), sizeof(double));
        double *tW = (double *)calloc((size_t)nb, sizeof(double));
        double *tO = (double *)calloc((size_t)nb, sizeof(double));
        uint64_t tk = 0;
        double *eta_p = NULL, *eta_q = NULL;
        int32_t *bins = NULL;
        int64_t cap_p = 0, cap_q = 0, cap_b = 0;
#pragma omp for schedule(dynamic, 16)
        for (int64_t k = 0; k < n_pairs; ++k) {
            int64_t p = pq[2 * k], q = pq[2 * k + 1];
            int64_t op = f->pix_off[p], oq = f->pix_off[q];
            int64_t np = f->pix_off[p + 1] - op, nq = f->pix_off[q + 1] - oq;
            if (np * np > cap_p) { free(eta_p); cap_p = np * np; eta_p = (double *)malloc(sizeof(double) * (size_t)cap_p); }
            if (nq * nq > cap_q) { free(eta_q); cap_q = nq * nq; eta_q = (double *)malloc(sizeof(double) * (size_t)cap_q); }
            if (np * nq > cap_b) { free(bins); cap_b = np * nq; bins = (int32_t *)malloc(sizeof(int32_t) * (size_t)cap_b); }
            if (orc_eta(np, f->w + op, f->loglam + op, eta_p) ||
                orc_eta(nq, f->w + oq, f->loglam + oq, eta_q)) {
#pragma omp atomic write
                bad = 1;
                continue;
            }
            double s, c;
            orc_pair_sc(f, p, q, &s, &c);
            for (int64_t i = 0; i < np; ++i)
                for (int64_t j = 0; j < nq; ++j)
                    bins[i * nq + j] = pix_bin(b, s, c, f->chi[op + i], f->chi[oq + j]);
            for (int64_t i = 0; i < np; ++i)
                for (int64_t j = 0; j < nq; ++j) {
                    int32_t A = bins[i * nq + j];
                    if (A < 0) continue;
                    if (!orc_keep(seed, op + i, oq + j, thr)) continue;
                    double om = f->w[op + i] * f->w[oq + j];
                    tW[A] += om;
                    ++tk;
                    double *row = tD + (int64_t)A * nb;
                    for (int64_t i2 = 0; i2 < np; ++i2) {
                        double e1 = om * eta_p[i * np + i2];
                        for (int64_t j2 = 0; j2 < nq; ++j2) {
                            int32_t B = bins[i2 * nq + j2];
                            double term = e1 * eta_q[j * nq + j2];
                            if (B >= 0) row[B] += term; else tO[A] += term;
                        }
                    }
                }
        }
#pragma omp critical
        {
            for (int64_t a = 0; a < nb * nb; ++a) Dn[a] += tD[a];
            for (int64_t a = 0; a < nb; ++a) { Wd[a] += tW[a]; if (Dover) Dover[a] += tO[a]; }
            kept += tk;
        }
        free(tD); free(tW); free(tO); free(eta_p); free(eta_q); free(bins);
    }
    if (n_kept) n_kept[0] = kept;
    if (D)
        for (int64_t A = 0; A < nb; ++A)
            for (int64_t B = 0; B < nb; ++B)
                D[A * nb + B] = (Wd[A] != 0.0) ? Dn[A * nb + B] / Wd[A] : 0.0;
    return bad;
}

/* ---- CROSS-CHECK ONLY (pin PD4): D through the rank-2 form of eta ----------- */
/*
 * eta_ii' = delta^K_ii' - a_i' - u_i g_i',  a = w/sum(w), u = L - Lbar,
 * g = w u / sum(w u^2).  Then for a kept pair (i,j), with H_xy[B] =
 * sum_{(i',j') in B} x_i' y_j':
 *   sum_{(i',j') in B} eta_ii' eta_jj' = [B == A]
 *      - sum_{j': bin(i,j')=B} (a_j' + u_j g_j') - sum_{i': bin(i',j)=B} (a_i' + u_i g_i')
 *      + H_aa[B] + u_j H_ag[B] + u_i H_ga[B] + u_i u_j H_gg[B].
 * Independent of the CUDA code; used to cross-check orc_dmat (PD4) and as the
 * declared fallback reference where the naive sum is too slow (DESIGN.md O-D4).
 */
int orc_dmat_collapsed(const orc_forests *f, const orc_binning *b, const int32_t *pq, int64_t n_pairs,
                       double reject_fraction, uint64_t seed,
                       double *Dn, double *Wd, uint64_t *n_kept)
{
    int64_t nb = (int64_t)b->n_par * b->n_perp;
    uint64_t thr = orc_mask_threshold(reject_fraction);
    memset(Dn, 0, sizeof(double) * (size_t)(nb * nb));
    memset(Wd, 0, sizeof(double) * (size_t)nb);
    uint64_t kept = 0;
    int bad = 0;
    /* per-pixel a, u, g for the whole catalogue */
    double *a = (double *)malloc(sizeof(double) * (size_t)f->n_pix);
    double *u = (double *)malloc(sizeof(double) * (size_t)f->n_pix);
    double *g = (double *)malloc(sizeof(double) * (size_t)f->n_pix);
    for (int64_t p = 0; p < f->n_forest; ++p) {
        int64_t o = f->pix_off[p], n = f->pix_off[p + 1] - o;
        long double sw = 0, swl = 0, v = 0;
        for (int64_t k = 0; k < n; ++k) { sw += f->w[o + k]; swl += (long double)f->w[o + k] * f->loglam[o + k]; }
        double lbar = (sw > 0) ? (double)(swl / sw) : 0.0;
        for (int64_t k = 0; k < n; ++k) { u[o + k] = f->loglam[o + k] - lbar; v += (long double)f->w[o + k] * u[o + k] * u[o + k]; }
        for (int64_t k = 0; k < n; ++k) {
            a[o + k] = (sw > 0) ? f->w[o + k] / (double)sw : NAN;
            g[o + k] = (v > 0) ? f->w[o + k] * u[o + k] / (double)v : NAN;
        }
    }
#pragma omp parallel
    {
        double *tD = (double *)calloc((size_t)(nb * nb), sizeof(double));
        double *tW = (double *)calloc((size_t)nb, sizeof(double));
        double *H = (double *)calloc((size_t)(4 * nb), sizeof(double));
        int32_t *support = (int32_t *)malloc(sizeof(int32_t) * (size_t)nb);
        char *seen = (char *)calloc((size_t)nb, 1);
        int32_t *bins = NULL; int64_t cap_b = 0;
        uint64_t tk = 0;
#pragma omp for schedule(dynamic, 16)
        for (int64_t k = 0; k < n_pairs; ++k) {
            int64_t p = pq[2 * k], q = pq[2 * k + 1];
            int64_t op = f->pix_off[p], oq = f->pix_off[q];
            int64_t np = f->pix_off[p + 1] - op, nq = f->pix_off[q + 1] - oq;
            if (np == 0 || nq == 0) continue;
            if (isnan(a[op]) || isnan(g[op]) || isnan(a[oq]) || isnan(g[oq])) {
#pragma omp atomic write
                bad = 1;
                continue;
            }
            if (np * nq > cap_b) { free(bins); cap_b = np * nq; bins = (int32_t *)malloc(sizeof(int32_t) * (size_t)cap_b); }
            double s, c;
            orc_pair_sc(f, p, q, &s, &c);
            int32_t n_sup = 0;                     /* distinct in-grid bins of this forest pair */
            for (int64_t i = 0; i < np; ++i)
                for (int64_t j = 0; j < nq; ++j) {
                    int32_t B = pix_bin(b, s, c, f->chi[op + i], f->chi[oq + j]);
                    bins[i * nq + j] = B;
                    if (B < 0) continue;
                    if (!seen[B]) { seen[B] = 1; support[n_sup++] = B; }
                    H[4 * B + 0] += a[op + i] * a[oq + j];
                    H[4 * B + 1] += a[op + i] * g[oq + j];
                    H[4 * B + 2] += g[op + i] * a[oq + j];
                    H[4 * B + 3] += g[op + i] * g[oq + j];
                }
            for (int64_t i = 0; i < np; ++i)
                for (int64_t j = 0; j < nq; ++j) {
                    int32_t A = bins[i * nq + j];
                    if (A < 0 || !orc_keep(seed, op + i, oq + j, thr)) continue;
                    double om = f->w[op + i] * f->w[oq + j];
                    double ui = u[op + i], uj = u[oq + j];
                    double *row = tD + (int64_t)A * nb;
                    tW[A] += om; ++tk;
                    row[A] += om;
                    for (int64_t j2 = 0; j2 < nq; ++j2) {
                        int32_t B = bins[i * nq + j2];
                        if (B >= 0) row[B] -= om * (a[oq + j2] + uj * g[oq + j2]);
                    }
                    for (int64_t i2 = 0; i2 < np; ++i2) {
                        int32_t B = bins[i2 * nq + j];
                        if (B >= 0) row[B] -= om * (a[op + i2] + ui * g[op + i2]);
                    }
                    for (int32_t t = 0; t < n_sup; ++t) {
                        int32_t B = support[t];
                        row[B] += om * (H[4 * B + 0] + uj * H[4 * B + 1] + ui * H[4 * B + 2] + ui * uj * H[4 * B + 3]);
                    }
                }
            for (int32_t t = 0; t < n_sup; ++t) {
                int32_t B = support[t];
                seen[B] = 0; H[4 * B] = H[4 * B + 1] = H[4 * B + 2] = H[4 * B + 3] = 0.0;
            }
        }
#pragma omp critical
        {
            for (int64_t x = 0; x < nb * nb; ++x) Dn[x] += tD[x];
            for (int64_t x = 0; x < nb; ++x) Wd[x] += tW[x];
            kept += tk;
        }
        free(tD); free(tW); free(H); free(bins); free(support); free(seen);
    }
    free(a); free(u); free(g);
    if (n_kept) n_kept[0] = kept;
    return bad;
}

/* ==========================================================================================
 * NEXT-4: brute-force anisotropic three-point correlation function, eq. 2.8:
 *     xi3_A = sum_A (d_i w_i)(d_j w_j)(d_k w_k) / sum_A w_i w_j w_k,   i, j, k in DISTINCT quasars,
 * binned in the five triangle variables of PAPER.md:108 and Fig. 2 / Fig. 5: the two
 * sides r1, r2 from a main vertex, the inner angle alpha (binned in cos alpha) and the angles theta1,
 * theta2 of the two sides to the line of sight.  "The same triangle is recorded ... depending on which
 * point is taken as the main vertex".
 *
 * The paper fixes neither the vertex convention, nor the line of sight, nor the flattening; the readings
 * (T1-T7), each operation one separately rounded binary64 operation, no FMA:
 *  T1 position of a pixel: X = (chi ux, chi uy, chi uz) (flat universe, comoving Cartesian).
 *  T2 every ORDERED triple (i; j, k) counts: i the main vertex, j the end of side 1, k the end of side 2,
 *     the three pixels in three distinct forests (so a triangle enters 6 times: 3 vertices x 2 orders).
 *  T3 side vectors d1 = X_j - X_i, d2 = X_k - X_i; r = sqrt(((dx dx) + (dy dy)) + (dz dz));
 *     a side takes part iff 0 < r < r_max.
 *  T4 line of sight = the unit vector u of the main vertex's forest;
 *     cos theta = (((dx ux) + (dy uy)) + (dz uz)) / r;   cos alpha = (((d1x d2x) + (d1y d2y)) + (d1z d2z)) / (r1 r2).
 *  T5 bins: b_r = (int)(r (n_r / r_max)) clamped to n_r - 1;
 *     b_theta = number of m in 1..n_theta-1 with cos theta <= C_m, C_m = cos(m pi / n_theta) -- equal steps in
 *     theta over [0, pi] without an arccos (libm's differs between host and device in the last bit); the
 *     table C is an INPUT computed once by the caller, like chi;
 *     b_alpha = (int)((cos alpha + 1) (n_cosa / 2)) clamped to [0, n_cosa - 1].
 *  T6 triangle index A = (((b_r1 n_r + b_r2) n_cosa + b_alpha) n_theta + b_theta1) n_theta + b_theta2.
 *  T7 sums: S3 += ((a_i a_j) a_k) with a = w d;  W3 += ((w_i w_j) w_k);  N3 += 1.
 * The forest-pair list pq (p < q) only has to hold every pair of forests with two pixels closer than
 * r_max (any superset gives the same sums); adjacency is taken from it in both directions. */
typedef struct { double r_max; int32_t n_r, n_theta, n_cosa; } orc_tri_binning;

static inline int tri_side(const orc_tri_binning *tb, const double *cosedge, const double xi[3], const double ui[3],
                           double chi_j, const double uj[3], double d[3], double *r, int32_t *b_r, int32_t *b_t)
{
    double xj0 = chi_j * uj[0], xj1 = chi_j * uj[1], xj2 = chi_j * uj[2];
    d[0] = xj0 - xi[0]; d[1] = xj1 - xi[1]; d[2] = xj2 - xi[2];
    double r2 = ((d[0] * d[0]) + (d[1] * d[1])) + (d[2] * d[2]);
    *r = sqrt(r2);
    if (!(*r > 0.0) || !(*r < tb->r_max)) return 0;
    double inv = (double)tb->n_r / tb->r_max;
    int32_t br = (int32_t)(*r * inv);
    if (br > tb->n_r - 1) br = tb->n_r - 1;
    double ct = (((d[0] * ui[0]) + (d[1] * ui[1])) + (d[2] * ui[2])) / *r;
    int32_t bt = 0;
    for (int32_t m = 0; m < tb->n_theta - 1; ++m) bt += (ct <= cosedge[m]) ? 1 : 0;
    *b_r = br; *b_t = bt;
    return 1;
}

int64_t orc_tri_nbins(const orc_tri_binning *tb)
{
    return (int64_t)tb->n_r * tb->n_r * tb->n_cosa * tb->n_theta * tb->n_theta;
}

void orc_xi3(const orc_forests *f, const orc_tri_binning *tb, const double *cosedge, const int32_t *pq, int64_t n_pairs,
             double *S3, double *W3, uint64_t *N3)
{
    int64_t nf = f->n_forest, nb = orc_tri_nbins(tb);
    /* adjacency in both directions from the pair list */
    int64_t *deg = (int64_t *)calloc((size_t)nf + 1, sizeof(int64_t));
    for (int64_t k = 0; k < n_pairs; ++k) { deg[pq[2 * k] + 1]++; deg[pq[2 * k + 1] + 1]++; }
    for (int64_t p = 0; p < nf; ++p) deg[p + 1] += deg[p];
    int32_t *adj = (int32_t *)malloc(sizeof(int32_t) * (size_t)(2 * n_pairs + 1));
    int64_t *cur = (int64_t *)malloc(sizeof(int64_t) * (size_t)(nf + 1));
    memcpy(cur, deg, sizeof(int64_t) * (size_t)(nf + 1));
    for (int64_t k = 0; k < n_pairs; ++k) {
        adj[cur[pq[2 * k]]++] = pq[2 * k + 1];
        adj[cur[pq[2 * k + 1]]++] = pq[2 * k];
    }
    long double *gS = (long double *)calloc((size_t)nb, sizeof(long double));
    long double *gW = (long double *)calloc((size_t)nb, sizeof(long double));
    memset(N3, 0, sizeof(uint64_t) * (size_t)nb);
    double nhalf = (double)tb->n_cosa / 2.0;
#pragma omp parallel
    {
        long double *tS = (long double *)calloc((size_t)nb, sizeof(long double));
        long double *tW = (long double *)calloc((size_t)nb, sizeof(long double));
        uint64_t *tN = (uint64_t *)calloc((size_t)nb, sizeof(uint64_t));
#pragma omp for schedule(dynamic, 1)
        for (int64_t p = 0; p < nf; ++p) {
            double ui[3] = { f->ux[p], f->uy[p], f->uz[p] };
            for (int64_t i = f->pix_off[p]; i < f->pix_off[p + 1]; ++i) {
                double xi[3] = { f->chi[i] * ui[0], f->chi[i] * ui[1], f->chi[i] * ui[2] };
                double ai = f->w[i] * f->delta[i], wi = f->w[i];
                for (int64_t eq = deg[p]; eq < deg[p + 1]; ++eq) {
                    int64_t q = adj[eq];
                    double uq[3] = { f->ux[q], f->uy[q], f->uz[q] };
                    for (int64_t j = f->pix_off[q]; j < f->pix_off[q + 1]; ++j) {
                        double d1[3], r1; int32_t br1, bt1;
                        if (!tri_side(tb, cosedge, xi, ui, f->chi[j], uq, d1, &r1, &br1, &bt1)) continue;
                        double aij = ai * (f->w[j] * f->delta[j]), wij = wi * f->w[j];
                        for (int64_t er = deg[p]; er < deg[p + 1]; ++er) {
                            int64_t r = adj[er];
                            if (r == q) continue;
                            double ur[3] = { f->ux[r], f->uy[r], f->uz[r] };
                            for (int64_t k = f->pix_off[r]; k < f->pix_off[r + 1]; ++k) {
                                double d2[3], r2; int32_t br2, bt2;
                                if (!tri_side(tb, cosedge, xi, ui, f->chi[k], ur, d2, &r2, &br2, &bt2)) continue;
                                double ca = (((d1[0] * d2[0]) + (d1[1] * d2[1])) + (d1[2] * d2[2])) / (r1 * r2);
                                int32_t ba = (int32_t)((ca + 1.0) * nhalf);
                                if (ba < 0) ba = 0;
                                if (ba > tb->n_cosa - 1) ba = tb->n_cosa - 1;
                                int64_t A = ((((int64_t)br1 * tb->n_r + br2) * tb->n_cosa + ba) * tb->n_theta + bt1) * tb->n_theta + bt2;
                                tS[A] += aij * (f->w[k] * f->delta[k]);
                                tW[A] += wij * f->w[k];
                                tN[A] += 1;
                            }
                        }
                    }
                }
            }
        }
#pragma omp critical
        for (int64_t a = 0; a < nb; ++a) { gS[a] += tS[a]; gW[a] += tW[a]; N3[a] += tN[a]; }
        free(tS); free(tW); free(tN);
    }
    for (int64_t a = 0; a < nb; ++a) { S3[a] = (double)gS[a]; W3[a] = (double)gW[a]; }
    free(gS); free(gW); free(deg); free(adj); free(cur);
}
