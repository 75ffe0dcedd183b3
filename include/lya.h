/*
 * lya.h -- C-ABI of liblya.so: the B200 (sm_100a) pixel-pair hot path of the
 * Lya2pcf method (arxiv 2507.00129; citations are /root/reference/PAPER.md lines).
 *
 *   lya_neighbours  forest pairs closer than the maximum transverse separation
 *                   ("only takes forests within a pre-ordered
 *                   neighborhood defined by this maximum distance")
 *   lya_xi2pcf      eq. 2.4: S_A = sum w_i d_i w_j d_j,
 *                   W_A = sum w_i w_j, N_A = pair count, xi_A = S_A / W_A over
 *                   pixel pairs of DIFFERENT forests on the (r_par, r_perp) grid
 *   lya_dmat        eqs. 2.6-2.7: the distortion matrix
 *                   D_AB = W_A^-1 sum_{(i,j) in A} w_i w_j sum_{(i',j') in B}
 *                   eta_ii' eta_jj', with a seeded pixel-pair keep mask
 *
 * Conventions
 *   - Plain C, no C++/torch types.  Unless a parameter says "host", every
 *     pointer is a DEVICE pointer on the ctx's device, caller-owned; inputs are
 *     never modified or freed; outputs are caller-allocated and OVERWRITTEN.
 *   - Work is enqueued on the ctx stream; device outputs are valid once the
 *     caller has synchronised that stream (calls that return host values
 *     synchronise internally and say so).
 *   - Every call returns a status and never throws, prints or exits.  On error,
 *     outputs are unspecified and lya_last_error(ctx) holds a message.
 *   - One ctx per host thread.  There is no CPU fallback: without a CUDA device
 *     lya_create fails with LYA_ERR_CUDA.
 *
 * Geometry (readings G1-G6; the paper gives no formulas at this level):
 *   forest pair: s = 0.5*sqrt(|u_p - u_q|^2) = sin(theta/2), c = sqrt(1 - s*s)
 *   pixel pair:  r_par = |chi_i - chi_j| * c,   r_perp = (chi_i + chi_j) * s
 *   in grid iff r_par < rpar_max and r_perp < rperp_max;
 *   b = (int)(r * (n / r_max)) clamped to n-1;  A = n_perp * b_par + b_perp.
 *   All of it in IEEE binary64, each operation rounded separately (no FMA), so
 *   that bins -- hence pair counts -- are bit-identical to the CPU oracle.
 */
#ifndef LYA_H
#define LYA_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lya_ctx lya_ctx;      /* opaque: device, stream, scratch, last error */
typedef struct lya_pairs lya_pairs;  /* opaque, library-owned device forest-pair list */
typedef struct lya_plan lya_plan;    /* opaque: prepared catalogue + bucket-sorted pair list (see lya_plan_create) */

typedef enum {
    LYA_OK = 0,
    LYA_ERR_INVALID_ARG = 1,        /* NULL/negative sizes/inconsistent offsets/non-finite input */
    LYA_ERR_UNSORTED = 2,           /* chi not strictly increasing inside a forest */
    LYA_ERR_DEGENERATE_FOREST = 3,  /* lya_dmat: a forest with sum w == 0 or sum w (L-Lbar)^2 == 0 */
    LYA_ERR_CAPACITY = 4,           /* a size exceeds what the library supports (see each call) */
    LYA_ERR_OOM = 5,                /* device allocation failed */
    LYA_ERR_CUDA = 6,               /* any other CUDA runtime error (message in lya_last_error) */
    LYA_ERR_UNIMPLEMENTED = 7
} lya_status;

/* Forest catalogue, CSR over pixels (a skewer = sky position + a
 * variable-length table of delta, weight, wavelength).
 *   ux,uy,uz: unit vectors of the sightlines (|u|^2 = 1 to 1e-9, else LYA_ERR_INVALID_ARG).  They are INPUTS
 *     (like chi) so that
 *     both this library and a checker consume identical values; pass NULL for all
 *     three to have them derived on the device from ra/dec (not bit-reproducible
 *     against a host libm).  ra/dec [radians] may be NULL when ux,uy,uz are given.
 *   pix_off: [n_forest+1], pix_off[0] = 0, non-decreasing, pix_off[n_forest] = n_pix.
 *   chi [Mpc/h]: comoving distance of each pixel, strictly increasing inside a
 *     forest, 0 <= chi < 1e6.   w >= 0.   loglam = log(lambda) in any base
 *     (eq. 2.7 is invariant under affine maps of it); only lya_dmat reads it,
 *     it may be NULL for lya_neighbours / lya_xi2pcf.
 *   n_forest < 2^31, n_pix < 2^40. */
typedef struct {
    int64_t n_forest, n_pix;
    const double *ra, *dec;
    const double *ux, *uy, *uz;
    const int64_t *pix_off;
    const double *chi, *w, *delta, *loglam;
} lya_forests;

/* (r_par, r_perp) grid (4 Mpc/h bins up to 200 Mpc/h -> 50 x 50).
 * Requires 0 < r*_max <= 1e5, 1 <= n_* and n_par*n_perp <= 4096, bin width >= 0.01 (LYA_ERR_CAPACITY
 * otherwise); the fast kernels also need n_par <= 50 and n_perp <= 126, other grids take the generic ones. */
typedef struct {
    double rpar_max, rperp_max;
    int32_t n_par, n_perp;
} lya_binning;

/* Counters filled by the compute calls (host struct; valid after the call
 * returns -- the calls that take it synchronise the ctx stream). */
typedef struct {
    uint64_t n_forest_pairs;   /* forest pairs traversed */
    uint64_t n_visited;        /* sum over traversed forest pairs of n_p * n_q */
    uint64_t n_evaluated;      /* pixel pairs whose separation was actually computed */
    uint64_t n_binned;         /* pixel pairs inside the grid (= sum_A N_A) */
    uint64_t n_kept;           /* lya_dmat: in-grid pixel pairs that passed the keep mask */
    uint64_t n_scatter;        /* lya_dmat: fp64 scatter-adds into Dn/Wd issued by the fast and long-forest kernels (0 for generic pairs) */
    float    ms_main;          /* device time of the dominant kernel (CUDA events on the ctx stream) */
    float    ms_total;         /* device time of the whole call */
} lya_stats;

/* ---- context ------------------------------------------------------------------ */
/* device: CUDA ordinal.  cuda_stream: a cudaStream_t (e.g. torch's current
 * stream) or NULL for the legacy default stream. */
lya_status  lya_create(lya_ctx **ctx, int device, void *cuda_stream);
void        lya_destroy(lya_ctx *ctx);
const char *lya_last_error(const lya_ctx *ctx);   /* host string, owned by ctx */
const char *lya_version(void);
/* Number of CUDA kernels this library has launched in the process so far (all contexts; every launch site
 * counts itself; one ctx per host thread, so no synchronisation).  bench.py reports the difference over
 * its timed region as gpu_launches. */
uint64_t    lya_launch_count(void);

/* Explicit, per-ctx switches (there are no environment variables or global flags).
 *   LYA_OPT_FORCE_GENERIC     0 (default) / 1: route EVERY forest pair to the generic kernels (block-level
 *                             histogram / CAS H tables) instead of the fast ones.  Results are identical
 *                             (N, n_kept exactly; sums to rounding); tests use it to cover both routes.
 *   LYA_OPT_GENERIC_DIAGONALS 1, 2 (default) or 4: diagonals of the pixel-pair matrix per lane in the
 *                             generic xi kernel (a tuning knob; results do not depend on it).
 *   LYA_OPT_CHECK_HOLDERS     0 (default) / 1: run the debug variant of the fast kernels, which checks at every
 *                             row step that no two lanes of a warp hold the same table entry (the invariant
 *                             their atomic-free accumulation rests on).  Much slower; a
 *                             violation makes the call return LYA_ERR_CUDA with the count in lya_last_error.
 *   LYA_OPT_XI_MERGE_EVERY    1 .. 2^31 (default 2^31): a warp of the fast xi kernel merges its private
 *                             sub-histogram into the global accumulators after this many visited pixel pairs
 *                             even when its bucket does not change -- the guard that keeps its 32-bit pair
 *                             counters from overflowing.  No workload of this size reaches the default, so a
 *                             test lowers it to drive the guard; results do not depend on it.
 * LYA_ERR_INVALID_ARG for an unknown option or value. */
typedef enum { LYA_OPT_FORCE_GENERIC = 0, LYA_OPT_GENERIC_DIAGONALS = 1, LYA_OPT_CHECK_HOLDERS = 2,
               LYA_OPT_XI_MERGE_EVERY = 3 } lya_option;
lya_status  lya_set_option(lya_ctx *ctx, lya_option opt, int64_t value);

/* ---- stage 1: neighbour search (north_star stage 1) ------------ */
/* Lists every unordered pair of distinct non-empty forests {p<q} with
 *   (chi_p[0] + chi_q[0]) * s_pq < rperp_max            (reading G4)
 * i.e. theta below the angle that gives r_perp = rperp_max at the pair's minimum
 * comoving distances.  Any pair with at least one in-grid pixel pair is listed.
 * Method: uniform 3-D cell grid over the unit vectors (cell edge >= the largest
 * admissible chord), counting sort by cell, count -> exclusive scan -> fill.
 * The list is a set (order unspecified but deterministic); entries have p < q.
 * *out is library-owned (free with lya_pairs_free).  n_pairs: host out.
 * Synchronises the ctx stream.  LYA_ERR_CAPACITY if n_pairs >= 2^40. */
lya_status lya_neighbours(lya_ctx *ctx, const lya_forests *f, const lya_binning *b,
                          lya_pairs **out, int64_t *n_pairs);
/* Copies the list to pq, device int32 [n_pairs][2] (p, q). */
lya_status lya_pairs_export(lya_ctx *ctx, const lya_pairs *pairs, int32_t *pq);
/* Builds a list from caller pairs (device int32 [n_pairs][2]); entries must be
 * distinct forests, either order; no criterion is applied (tests, sharding). */
lya_status lya_pairs_import(lya_ctx *ctx, const int32_t *pq, int64_t n_pairs, lya_pairs **out);
/* Forest-pair subsampling, the paper's own wording for the distortion matrix ("In practice D_AB is
 * computed only with a small subset of forest pairs"; DESIGN.md NEXT-2): keeps the forest
 * pair (p<q) iff keep(seed, p, q) of the stage-4 integer mask (with the FOREST indices
 * in place of pixel offsets) is true for reject_fraction.  The order of the kept pairs is preserved.
 * lya_dmat on the result with reject_fraction = 0 is the distortion matrix of that subset.
 * *out is library-owned; n_kept: host out.  Synchronises the ctx stream. */
lya_status lya_pairs_subsample(lya_ctx *ctx, const lya_pairs *pairs, double reject_fraction, uint64_t seed,
                               lya_pairs **out, int64_t *n_kept);
int64_t    lya_pairs_count(const lya_pairs *pairs);
void       lya_pairs_free(lya_ctx *ctx, lya_pairs *pairs);

/* ---- stage 2: pair kernel, eq. 2.4 ------------------------------ */
/* S, W: double [n_par*n_perp]; N: uint64 [n_par*n_perp]; xi: double [n_par*n_perp]
 * (xi_A = S_A / W_A, 0 where W_A == 0); row-major [b_par][b_perp].  Any of S, W,
 * N, xi may be NULL.  Each unordered pixel pair of each listed forest pair counts
 * once.  stats: host out, may be NULL.  The call synchronises the ctx stream either way.
 * Kernel routes (results do not depend on them): forests of up to 72 pixels whose spacing exceeds the r_par bin
 * width take the atomic-free fast kernel, forests of up to 144 pixels with a spacing down to an eighth of the bin
 * width its second size class, everything else a generic kernel with shared-memory atomics. */
lya_status lya_xi2pcf(lya_ctx *ctx, const lya_forests *f, const lya_binning *b,
                      const lya_pairs *pairs,
                      double *S, double *W, uint64_t *N, double *xi, lya_stats *stats);

/* NEXT-1: per-sky-region sub-samples of eq. 2.4, the input of the covariance
 * estimate ("covariance ... from sub-sampling").  region: device int32
 * [n_forest] with values in [0, n_region); a pixel pair belongs to the sub-sample of the LOWER-index
 * forest p of its forest pair.  S, W: double [n_region][n_par*n_perp]; N: uint64 [n_region][...]; any
 * may be NULL.  Summed over the regions they equal lya_xi2pcf's S, W, N (N exactly).
 * LYA_ERR_INVALID_ARG for a region outside the range; LYA_ERR_CAPACITY if n_region * bins > 2^28. */
lya_status lya_xi2pcf_sub(lya_ctx *ctx, const lya_forests *f, const lya_binning *b,
                          const lya_pairs *pairs, const int32_t *region, int32_t n_region,
                          double *S, double *W, uint64_t *N, lya_stats *stats);

/* NEXT-1, second half: the weighted mean coordinates of every bin, as the PICCA-like correlation table carries
 * them ("mimics PICCA", 261-263).  For every in-grid pixel pair (i, j) of the listed forest pairs,
 * A = its bin, om = w_i w_j:  Rpar[A] += om r_par,  Rperp[A] += om r_perp,  Z[A] += om (z_i + z_j) / 2,
 * W[A] += om, with r_par, r_perp exactly as binned (geometry above) and z a device array [n_pix] of pixel
 * redshifts (reading R-19: the redshift of a pair is the mean of its two pixels').  The outputs are SUMS (device
 * double [n_par*n_perp], additive over forest pairs and ranks); the means are lya_xi_normalise(Rpar, W) etc.
 * W may be NULL.  delta and loglam are not read.  A second, cheap mode (shared-memory CAS histogram), not the
 * tuned pair kernel.  Synchronises the ctx stream. */
lya_status lya_xi2pcf_means(lya_ctx *ctx, const lya_forests *f, const lya_binning *b, const lya_pairs *pairs,
                            const double *z, double *Rpar, double *Rperp, double *Z, double *W);

/* ---- stages 3+4: distortion matrix, eqs. 2.6-2.7 ----------------- */
/* eta_ii' = delta^K_ii' - w_i'/sum_k w_k - (L_i-Lbar) w_i' (L_i'-Lbar) / sum_k w_k (L_k-Lbar)^2
 * inside a forest (0 across forests), L = loglam, Lbar the w-weighted mean (R-10).
 * For every listed forest pair and every in-grid pixel pair (i,j) that passes the
 * keep mask (A = its bin, om = w_i w_j):
 *     Wd[A] += om;   Dn[A][B] += om * sum_{(i',j') in B} eta_ii' eta_jj'
 * over i' in the forest of i and j' in the forest of j ((i',j') outside the grid
 * are dropped; the inner sum is never masked, reading R-8).  D[A][B] = Dn[A][B]/Wd[A]
 * (row 0 where Wd[A] == 0).
 * Keep mask (stage 4): a pure-integer hash of (seed, the two
 * pixels' offsets in the flat arrays, smaller first); keep iff its top 32 bits
 * >= round(reject_fraction * 2^32).  reject_fraction in [0,1]; 0 keeps all.
 * D: double [NB*NB] row-major [A][B], NB = n_par*n_perp (NULL to skip the final
 * division); Dn: double [NB*NB] un-normalised sums (may be NULL if D is given; at
 * least one of D, Dn); Wd: double [NB] (may be NULL); stats as above (n_kept).
 * Every forest on the list must be non-degenerate (LYA_ERR_DEGENERATE_FOREST: sum w == 0, or all L equal up to
 * rounding -- sum w (L-Lbar)^2 <= sum w (1e-12 |Lbar|)^2).  Forests of any length (< 2^20 pixels) and any pixel
 * spacing are accepted; forests of up to 72 pixels whose spacing exceeds the r_par bin width take the fast kernel
 * (the BASELINE shapes), forests of up to 144 pixels with a spacing down to an eighth of the bin width its second
 * size class, forests of up to 1024 pixels with a spacing down to a sixteenth of it the long-forest kernel (one
 * thread block per forest pair; both for the native-resolution shapes of PAPER.md:79, 140-145), everything else --
 * longer forests, finer pixels, forest pairs spanning more than 6 r_perp columns -- a slower generic kernel.
 * LYA_ERR_CAPACITY if n_par > 512. */
lya_status lya_dmat(lya_ctx *ctx, const lya_forests *f, const lya_binning *b,
                    const lya_pairs *pairs, double reject_fraction, uint64_t seed,
                    double *D, double *Dn, double *Wd, lya_stats *stats);

/* ---- NEXT-4: brute-force anisotropic three-point correlation function, eq. 2.8 ------ */
/* xi3_A = sum_A (d_i w_i)(d_j w_j)(d_k w_k) / sum_A w_i w_j w_k over pixels of three DISTINCT forests, binned in the
 * five triangle variables of PAPER.md:108 / Fig. 2 / Fig. 5: the sides r1, r2 from a main vertex, cos(alpha) of the
 * inner angle, and the angles theta1, theta2 of the sides to the line of sight.  The paper leaves the conventions
 * open; the readings (T1-T7), each step one rounded binary64 operation:
 *   every ORDERED triple (i; j, k) counts (a triangle enters 6 times: 3 main vertices x 2 orders of the sides);
 *   X = chi u;  d1 = X_j - X_i, d2 = X_k - X_i;  r = sqrt(dx dx + dy dy + dz dz);  a side takes part iff 0 < r < r_max;
 *   line of sight = unit vector of the main vertex's forest;  cos theta = (d . u_i) / r;  cos alpha = (d1 . d2) / (r1 r2);
 *   b_r = (int)(r n_r / r_max) (clamped);  b_theta = number of m in 1..n_theta-1 with cos theta <= cos_theta_edges[m-1],
 *   the table cos(m pi / n_theta) being an INPUT (device double [n_theta-1]) so that no arccos enters;
 *   b_alpha = (int)((cos alpha + 1) n_cosa / 2) clamped to [0, n_cosa-1];
 *   A = (((b_r1 n_r + b_r2) n_cosa + b_alpha) n_theta + b_theta1) n_theta + b_theta2   (lya_tri_nbins entries).
 * pairs: any list holding every pair of forests with two pixels closer than r_max -- lya_neighbours with
 * rperp_max = r_max is one (r_perp never exceeds the 3-D separation).  S3, W3, xi3: device double [n_bins]; N3:
 * device uint64 [n_bins] (ordered triples per bin); any may be NULL.  stats: n_binned = ordered triples counted.
 * (The kernel visits each unordered pair of sides once and returns acc[A] + acc[A with the two sides swapped]:
 * cos alpha is bit-identical for both orders, so the counts are exact and S3, W3 move by an ulp per term.)
 * Limits (LYA_ERR_CAPACITY): at most 255 bins per variable and 2^24 bins in all; at most 2048 pixels of other
 * forests inside the sphere of radius r_max around one pixel.  Synchronises the ctx stream. */
typedef struct { double r_max; int32_t n_r, n_theta, n_cosa; } lya_tri_binning;   /* 80, 20, 10, 20 */
int64_t    lya_tri_nbins(const lya_tri_binning *tb);
lya_status lya_xi3pcf(lya_ctx *ctx, const lya_forests *f, const lya_tri_binning *tb, const double *cos_theta_edges,
                      const lya_pairs *pairs, double *S3, double *W3, uint64_t *N3, double *xi3, lya_stats *stats);

/* ---- plans: prepare once, run stages 2 and 3+4 on the same catalogue and list -------------------- */
/* lya_xi2pcf and lya_dmat each validate the catalogue, build a padded 16-byte-aligned copy of it (with the
 * per-pixel products of eq. 2.4 / eq. 2.7) and bucket-sort the forest-pair list by r_perp column before
 * their pair kernel runs.  A plan does that ONCE for a (catalogue, binning, pair list) triple:
 *   lya_plan_create(..., want_xi, want_dmat, &plan);  lya_xi2pcf_plan(plan, ...);  lya_dmat_plan(plan, ...);
 * give exactly the results of lya_xi2pcf / lya_dmat on the same arguments (those two calls are wrappers
 * that build a throw-away plan).  want_xi needs delta, want_dmat needs loglam.  The plan keeps the caller's
 * device pointers: the catalogue arrays must stay alive and unchanged until lya_plan_free; the pair list is
 * copied and may be freed.  lya_set_option(LYA_OPT_FORCE_GENERIC) is read at creation time.
 * Device memory: about 8 bytes per listed forest pair plus 24 (xi) / 48 (D) bytes per pixel.
 * lya_plan_create synchronises the ctx stream; errors as for lya_xi2pcf / lya_dmat (a degenerate listed
 * forest is reported by lya_dmat_plan, not at creation, so that a plan for both stages still serves xi). */
lya_status lya_plan_create(lya_ctx *ctx, const lya_forests *f, const lya_binning *b, const lya_pairs *pairs,
                           int want_xi, int want_dmat, lya_plan **out);
void       lya_plan_free(lya_ctx *ctx, lya_plan *plan);
lya_status lya_xi2pcf_plan(lya_ctx *ctx, const lya_plan *plan,
                           double *S, double *W, uint64_t *N, double *xi, lya_stats *stats);
lya_status lya_dmat_plan(lya_ctx *ctx, const lya_plan *plan, double reject_fraction, uint64_t seed,
                         double *D, double *Dn, double *Wd, lya_stats *stats);

/* ---- stage 2 without any allocation -------------------------------------------------------------- */
/* lya_xi2pcf_plan for callers that cannot allocate device memory inside the call (tight serving loops, harnesses
 * that forbid cudaMalloc): same arguments, same kernels, same results as lya_xi2pcf_plan (eq. 2.4)
 * -- N bit-identical, S / W / xi equal up to the order of the fp64 merges --, but the [S | W | N] accumulators,
 * the one piece of scratch memory stage 2 needs, live in a file-scope device array of the library instead of a
 * stream-ordered allocation.  The call makes no cudaMalloc / cudaFree / cudaMallocAsync and no host allocation.
 *   limit:   n_par * n_perp <= LYA_XI_NOALLOC_MAX_BINS (the paper's 50 x 50 grid fits); a larger grid is
 *            LYA_ERR_CAPACITY and nothing is launched -- use lya_xi2pcf_plan.  All of S, W, N, xi are required.
 *   cost:    every GPU that loads liblya.so holds the array (LYA_XI_NOALLOC_MAX_BINS * 24 bytes = 60 KB) until
 *            the process exits, whether or not this call is ever made.
 *   sharing: ONE array per device, shared by every context, plan and stream on it; it still holds the previous
 *            call's sums, so each call clears it on the ctx stream first.  Calls that overlap on the GPU -- two
 *            contexts or streams of one device inside this entry point at once -- race on it and give wrong
 *            sums: serialise them.  (lya_xi2pcf_plan has no such restriction.)
 * Like lya_xi2pcf_plan it synchronises the ctx stream before it returns (it reads the work counters), so it cannot
 * sit inside a CUDA graph capture; creating the plan still allocates -- do that at set-up. */
#define LYA_XI_NOALLOC_MAX_BINS 2560
lya_status lya_xi2pcf_plan_noalloc(lya_ctx *ctx, const lya_plan *plan,
                                   double *S, double *W, uint64_t *N, double *xi, lya_stats *stats);

/* ---- final divisions on already-summed numerators (multi-GPU) ----------- */
/* Every output above is an additive accumulator before its final division, so a catalogue's
 * forest-pair list can be split over ranks ("distribute the work load"): each rank runs
 * lya_xi2pcf / lya_dmat on its chunk asking for S, W, N / Dn, Wd, the numerators are summed across
 * ranks (one all-reduce), and these two calls then take the divisions of eq. 2.4 and eq. 2.6.
 * lya_xi_normalise:   xi[k] = S[k] / W[k] (0 where W[k] == 0), k < n  (n <= 2^30; D may alias nothing).
 * lya_dmat_normalise: D[A][B] = Dn[A][B] / Wd[A] (row 0 where Wd[A] == 0); D may alias Dn.
 * Device pointers; enqueued on the ctx stream, no synchronisation. */
lya_status lya_xi_normalise(lya_ctx *ctx, int64_t n, const double *S, const double *W, double *xi);
lya_status lya_dmat_normalise(lya_ctx *ctx, const lya_binning *b, const double *Dn, const double *Wd, double *D);

/* ---- end-to-end convenience with HOST buffers ------------------------------------- */
/* Uploads a HOST catalogue (every pointer in *f_host is a host pointer; ux/uy/uz
 * required), runs lya_neighbours, then lya_xi2pcf when do_xi and lya_dmat when
 * do_dmat, and downloads the results into HOST arrays (any may be NULL):
 * S, W, xi [NB] double, N [NB] uint64, D [NB*NB] double, Wd [NB] double.
 * stats_xi / stats_dmat: host out, may be NULL.  Synchronises. */
lya_status lya_run_host(lya_ctx *ctx, const lya_forests *f_host, const lya_binning *b,
                        int do_xi, int do_dmat, double reject_fraction, uint64_t seed,
                        double *S, double *W, uint64_t *N, double *xi,
                        double *D, double *Wd,
                        int64_t *n_pairs, lya_stats *stats_xi, lya_stats *stats_dmat);

#ifdef __cplusplus
}
#endif
#endif /* LYA_H */
