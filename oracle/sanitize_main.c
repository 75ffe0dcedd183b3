/* sanitize_main.c -- TEST INFRASTRUCTURE: drives every entry point of lya_oracle.c once on a small seeded
 * catalogue so that the oracle can be run under -fsanitize=address,undefined (
 * tests/test_oracle_sanitizers.py builds and runs it).  It checks nothing numerically (the pins do that):
 * a clean exit without a sanitizer report is the result. */
#include "lya_oracle.c"

static double lcg(unsigned long long *s)
{
    *s = *s * 6364136223846793005ULL + 1442695040888963407ULL;
    return (double)(*s >> 11) / 9007199254740992.0;
}

int main(void)
{
    enum { NF = 24 };
    unsigned long long seed = 2507001290ULL;
    int64_t off[NF + 1];
    off[0] = 0;
    for (int p = 0; p < NF; ++p) off[p + 1] = off[p] + (p == 5 ? 0 : (p == 6 ? 1 : 3 + (int)(lcg(&seed) * 20)));
    int64_t npix = off[NF];
    double *ux = malloc(sizeof(double) * NF), *uy = malloc(sizeof(double) * NF), *uz = malloc(sizeof(double) * NF);
    double *chi = malloc(sizeof(double) * npix), *w = malloc(sizeof(double) * npix), *dl = malloc(sizeof(double) * npix),
           *ll = malloc(sizeof(double) * npix), *z = malloc(sizeof(double) * npix);
    for (int p = 0; p < NF; ++p) {
        double ra = 0.03 * lcg(&seed), dec = 0.03 * lcg(&seed) - 0.015;
        ux[p] = cos(dec) * cos(ra); uy[p] = cos(dec) * sin(ra); uz[p] = sin(dec);
        double c = 3600.0 + 300.0 * lcg(&seed);
        for (int64_t k = off[p]; k < off[p + 1]; ++k) {
            c += 2.0 + 5.0 * lcg(&seed);
            chi[k] = c; w[k] = 0.5 + lcg(&seed); dl[k] = lcg(&seed) - 0.5; ll[k] = 3.55 + 1e-3 * (double)(k - off[p]);
            z[k] = 2.0 + 1e-3 * (double)(k - off[p]);
        }
    }
    orc_forests f = { NF, npix, ux, uy, uz, off, chi, w, dl, ll };
    orc_binning b = { 200.0, 200.0, 50, 50 };
    int32_t *pq = malloc(sizeof(int32_t) * 2 * NF * NF);
    int64_t n_all = orc_pairs_all(NF, pq);
    int64_t n_b = orc_pairs_brute(&f, &b, pq);
    int32_t *pq2 = malloc(sizeof(int32_t) * 2 * NF * NF);
    int64_t n_w = orc_pairs_window(&f, &b, pq2, (int64_t)NF * NF);
    int nb = 2500;
    double *S = calloc(nb, 8), *W = calloc(nb, 8), *xi = calloc(nb, 8), *Sa = calloc(nb, 8), *Q = calloc(nb, 8);
    uint64_t *N = calloc(nb, 8), n_out = 0;
    orc_xi(&f, &b, pq, n_b, S, W, N, xi, Sa, Q, &n_out);
    double *R1 = calloc(nb, 8), *R2 = calloc(nb, 8), *Z = calloc(nb, 8), *Wm = calloc(nb, 8);
    orc_xi_means(&f, &b, pq, n_b, z, R1, R2, Z, Wm);
    /* D: forests with fewer than 2 pixels are degenerate for eq. 2.7 -- keep pairs of healthy forests only */
    int64_t n_d = 0;
    for (int64_t k = 0; k < n_b; ++k) {
        int p = pq[2 * k], q = pq[2 * k + 1];
        if (off[p + 1] - off[p] >= 2 && off[q + 1] - off[q] >= 2) { pq2[2 * n_d] = p; pq2[2 * n_d + 1] = q; ++n_d; }
    }
    double *Dn = calloc((size_t)nb * nb, 8), *Wd = calloc(nb, 8), *Do = calloc(nb, 8);
    uint64_t n_kept = 0;
    int rc = orc_dmat(&f, &b, pq2, n_d, 0.5, 12345ULL, Dn, Wd, Do, &n_kept, NULL);
    double *Dc = calloc((size_t)nb * nb, 8), *Wc = calloc(nb, 8);
    uint64_t n_kept_c = 0;
    int rc2 = orc_dmat_collapsed(&f, &b, pq2, n_d, 0.5, 12345ULL, Dc, Wc, &n_kept_c);
    /* 3PCF on a coarse triangle grid (4 x 4 x 4 x 3 x 3 bins) */
    orc_tri_binning tb = { 80.0, 4, 3, 4 };
    double cosedge[2] = { 0.5, -0.5 };
    int64_t ntb = orc_tri_nbins(&tb);
    double *S3 = calloc((size_t)ntb, 8), *W3 = calloc((size_t)ntb, 8);
    uint64_t *N3 = calloc((size_t)ntb, 8);
    orc_xi3(&f, &tb, cosedge, pq, n_b, S3, W3, N3);
    free(S3); free(W3); free(N3);
    double eta[9 * 9];
    int rc3 = orc_eta(9, w, ll, eta);
    printf("sanitize_main: %lld all, %lld listed (%lld by the window), %llu out of grid, %llu kept (%llu), rc %d %d %d, thr %llu, keep %d\n",
           (long long)n_all, (long long)n_b, (long long)n_w, (unsigned long long)n_out, (unsigned long long)n_kept,
           (unsigned long long)n_kept_c, rc, rc2, rc3, (unsigned long long)orc_mask_threshold(0.99), orc_keep(1, 2, 3, 100));
    free(ux); free(uy); free(uz); free(chi); free(w); free(dl); free(ll); free(z); free(pq); free(pq2);
    free(S); free(W); free(xi); free(Sa); free(Q); free(N); free(R1); free(R2); free(Z); free(Wm);
    free(Dn); free(Wd); free(Do); free(Dc); free(Wc);
    return (n_b == n_w && n_kept == n_kept_c && rc == 0 && rc2 == 0 && rc3 == 0) ? 0 : 1;
}
