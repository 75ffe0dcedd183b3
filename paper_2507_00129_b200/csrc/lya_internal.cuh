// lya_internal.cuh -- shared declarations of liblya.so's translation units.
// (CUDA path only; the CPU oracle under oracle/ shares nothing with this.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include "../../include/lya.h"

#define LYA_CHI_MAX 1.0e6          // inputs must satisfy 0 <= chi < LYA_CHI_MAX
#define LYA_CHI_SENTINEL 1.0e7     // padding pixels: far outside any grid, still < 2^32 bins
#define LYA_MAX_BINS 4096

struct lya_ctx {
    int device;
    cudaStream_t stream;
    char err[512];
    int sm_count;
    // small persistent device scratch
    unsigned long long *d_counters;   // [16] work counters / flags
    int force_generic;                // LYA_OPT_FORCE_GENERIC: route every pair to the generic kernels
    int check_holders;                // LYA_OPT_CHECK_HOLDERS: debug variant of the fast kernels that asserts the one-holder invariant
    unsigned long long xi_merge_every; // LYA_OPT_XI_MERGE_EVERY: visited pairs between forced merges of a warp's sub-histogram
    int generic_diagonals;            // LYA_OPT_GENERIC_DIAGONALS: diagonals per lane of the generic xi kernel (1, 2, 4)
    cudaEvent_t ev[4];
    int use_pool;                     // scratch from the stream-ordered allocator (memory pools supported)
};

struct lya_pairs {
    int64_t n;
    int32_t *pq;       // device [n][2], p < q
    int max_len_hint;  // 0 = unknown
};

// device-visible error codes written by validation kernels (atomicMax)
enum { LYA_DEV_OK = 0, LYA_DEV_BAD_OFFSETS = 1, LYA_DEV_NONFINITE = 2, LYA_DEV_UNSORTED = 3,
       LYA_DEV_BAD_PAIR = 4, LYA_DEV_DEGENERATE = 5, LYA_DEV_TOO_LONG = 6 };

// process-wide count of kernel launches made by the library (lya_launch_count): every launch site notes itself
extern unsigned long long g_lya_launches;
static inline void lya_note_launch() { ++g_lya_launches; }

// Device scratch comes from CUDA's stream-ordered allocator on the ctx stream: the device's default memory pool
// keeps freed blocks (release threshold raised in lya_create), so the multi-GB pair lists and catalogue copies of
// one step are re-used by the next instead of being mapped and unmapped every call (0.3 s per step at configs[4]).
// lya_enter(ctx) is called by every entry point: it selects the device and makes the ctx stream the thread's
// allocation stream.
extern thread_local cudaStream_t tl_lya_stream;
extern thread_local bool tl_lya_pool;
cudaError_t lya_enter(lya_ctx *ctx);
template <class T> static inline cudaError_t lya_malloc(T **p, size_t bytes)
{
    return tl_lya_pool ? cudaMallocAsync((void **)p, bytes ? bytes : 1, tl_lya_stream) : cudaMalloc((void **)p, bytes ? bytes : 1);
}
static inline cudaError_t lya_free(void *p)
{
    if (!p) return cudaSuccess;
    return tl_lya_pool ? cudaFreeAsync(p, tl_lya_stream) : cudaFree(p);
}

lya_status lya_fail(lya_ctx *ctx, lya_status st, const char *fmt, ...);
lya_status lya_cuda_fail(lya_ctx *ctx, cudaError_t e, const char *what);
lya_status lya_check_binning(lya_ctx *ctx, const lya_binning *b);
lya_status lya_check_forests_host(lya_ctx *ctx, const lya_forests *f, bool need_u, bool need_delta, bool need_loglam);
// device-side validation of the catalogue (offsets, finiteness, monotone chi, w >= 0).
// Returns LYA_OK or the matching error; max forest length through *max_len.  Synchronises.
lya_status lya_validate_forests(lya_ctx *ctx, const lya_forests *f, bool need_delta, bool need_loglam,
                                int *max_len);

struct BinParams;
// ---- prepared catalogue (prep.cu): padded, 16-byte aligned SoA copy of the forests ----
// Every forest starts at an even offset and is padded to an even length, so each
// sub-array of a forest can be moved with 16-byte vector loads.  Pad pixels hold
// chi = LYA_CHI_SENTINEL and 0 elsewhere (never inside any grid).
struct __align__(16) ForestHead {   // 80 bytes, one per forest
    double ux, uy, uz;              // sightline unit vector
    double dmin;                    // smallest chi spacing inside the forest (1e300 if < 2 pixels)
    double chi0, chi1;              // first / last pixel (valid when len > 0)
    long long off;                  // offset of the forest in the packed arrays (even)
    long long pix0;                 // offset of the forest in the caller's flat arrays (stage-4 pixel ids)
    int len;                        // pixels
    int flags;                      // bit 0: degenerate for eq. 2.7 (sum w == 0 or sum w u^2 == 0)
};
struct LyaPrep {
    int64_t n_forest, n_pack;
    ForestHead *head;               // [n_forest]
    double *w;                      // [n_pack]
    double *chi, *a;                // xi: chi, w * delta
    double2 *ce;                    // dmat: (chi, ea) interleaved, ea = w / sum w            (eq. 2.7)
    double *eg, *u;                 // dmat: eg = w u / sum w u^2, u = L - Lbar
    void *base;                     // single allocation behind all of the above
    int max_len;
};
// Builds the prepared catalogue on the ctx stream (no host synchronisation except the
// one that returns n_pack).  want_xi -> a;  want_dmat -> u, ea, eg.
lya_status lya_prep_build(lya_ctx *ctx, const lya_forests *f, bool want_xi, bool want_dmat, LyaPrep *out);
void lya_prep_free(LyaPrep *p);

// ---- pair bucketing (prep.cu) -----------------------------------------------------------
// Stable counting sort of the forest-pair list by the r_perp column of the pair's first
// pixel pair (c_first).  Keys: 0..n_perp-1 = class-0 fast pairs (forests of up to LYA_FAST_TILE pixels whose
// spacing exceeds the r_par bin width; bins in columns [c_first, c_first + LYA_NCOL)); n_perp..2 n_perp-1 =
// class-1 fast pairs (up to LYA_FAST_TILE2 pixels, any spacing down to bin width / 8: the D kernel's second
// size class; the xi kernel sends them to its generic kernel); 2 n_perp = pairs for the generic kernels (longer
// forests, wider column span); 2 n_perp + 1 = pairs with nothing inside the grid.
#define LYA_NCOL 6                  // r_perp columns of a warp-private sub-histogram
#define LYA_FAST_TILE 72            // longest forest the class-0 fast kernels stage in one piece
#define LYA_FAST_TILE2 144          // same for class 1 (native-resolution shapes, DESIGN.md NEXT-3)
#define LYA_DS_MAX 8                // largest diagonal stride (bin width / pixel spacing, rounded up) of class 1
#define LYA_LONG_TILE 1024          // longest forest of the long-forest D kernel (one CTA per forest pair, dmat_long.cuh)
#define LYA_DS_MAX_LONG 16          // its largest diagonal stride (long rows keep the lanes busy at larger strides)
// Bucket keys of the sorted forest-pair list: [0, n_perp) class 0 by first column, [n_perp, 2 n_perp) class 1 by
// first column, then one key each for the long-forest D kernel, the generic kernels and the pairs with nothing in the grid.
#define LYA_KEY_LONG(n_perp) (2 * (n_perp))
#define LYA_KEY_GENERIC(n_perp) (2 * (n_perp) + 1)
#define LYA_KEY_SKIP(n_perp) (2 * (n_perp) + 2)
#define LYA_N_KEYS(n_perp) (2 * (n_perp) + 3)
struct LyaBuckets {
    int32_t *pq;                    // device [n][2], sorted by key (stable)
    int64_t n;
    int64_t n_fast, n_fast2, n_long, n_generic, n_skip;   // sizes of the five ranges of the sorted list, in this order
    unsigned long long visited;     // sum n_p * n_q over the whole list
    int bad_pair;                   // LYA_DEV_BAD_PAIR: a pair outside [0, n_forest); LYA_DEV_DEGENERATE: a listed degenerate forest
};
lya_status lya_bucket_pairs(lya_ctx *ctx, const LyaPrep *prep, const BinParams *bp, const lya_pairs *pairs,
                            int force_generic, LyaBuckets *out);
void lya_buckets_free(LyaBuckets *b);

// exclusive scan: in (u32 [n]) -> out (u64 [n+1], out[n] = total); tmp: ceil(n/2048)+2 u64
cudaError_t lya_exclusive_scan(const unsigned *in, unsigned long long *out, int64_t n, unsigned long long *tmp,
                               cudaStream_t s);

#define LYA_CUDA(call)                                                          \
    do {                                                                        \
        cudaError_t e__ = (call);                                               \
        if (e__ != cudaSuccess) return lya_cuda_fail(ctx, e__, #call);          \
    } while (0)

// Binning constants handed to kernels.
struct BinParams {
    double rpar_max, rperp_max;
    double inv_par, inv_perp;     // n / r_max
    int n_par, n_perp;
    int pow2;                     // both inverse widths are exact powers of two
};
static inline bool lya_is_pow2(double x)
{
    int e;
    return x > 0 && frexp(x, &e) == 0.5;
}
static inline BinParams lya_make_binparams(const lya_binning *b)
{
    BinParams bp;
    bp.rpar_max = b->rpar_max; bp.rperp_max = b->rperp_max;
    bp.n_par = b->n_par; bp.n_perp = b->n_perp;
    bp.inv_par = (double)b->n_par / b->rpar_max;
    bp.inv_perp = (double)b->n_perp / b->rperp_max;
    bp.pow2 = lya_is_pow2(bp.inv_par) && lya_is_pow2(bp.inv_perp) &&
              bp.inv_par * b->rpar_max == (double)b->n_par && bp.inv_perp * b->rperp_max == (double)b->n_perp;
    return bp;
}

// ---- plan (prep.cu): everything the pair kernels need that depends only on (catalogue, binning, pair list):
// the validated catalogue, its padded copy and the bucket-sorted forest-pair list.  Built once, used by
// lya_xi2pcf_plan / lya_dmat_plan any number of times (lya_xi2pcf / lya_dmat build a throw-away one).
#define LYA_FAST_NPAR_MAX 50         // r_par rows a warp-private table holds (both fast kernels)
struct lya_plan {
    lya_forests f;                  // the caller's arrays (must stay alive and unchanged while the plan is used)
    lya_binning b;
    BinParams bp;
    bool has_xi, has_dmat;          // which catalogue arrays were prepared
    bool use_fast;                  // bucketed list + fast kernels (else: every pair through the generic kernels)
    LyaPrep prep;
    LyaBuckets bk;                  // use_fast: sorted list [fast | generic | nothing in grid]
    int32_t *pq;                    // !use_fast: a copy of the pair list
    int64_t n_pairs;
    unsigned long long visited;     // sum n_p n_q over the list (use_fast)
    int listed_degenerate;          // has_dmat: a listed forest is degenerate for eq. 2.7
    int max_len;
};

#ifdef __CUDACC__
// ---- geometry, one separately rounded binary64 operation each (readings G2-G6) ----
// (explicit _rn intrinsics are never contracted into FMAs by nvcc)
__device__ __forceinline__ void lya_pair_sc(double uxp, double uyp, double uzp,
                                            double uxq, double uyq, double uzq, double &s, double &c)
{
    double dx = __dsub_rn(uxp, uxq), dy = __dsub_rn(uyp, uyq), dz = __dsub_rn(uzp, uzq);
    double h2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    s = __dmul_rn(0.5, __dsqrt_rn(h2));
    c = __dsqrt_rn(__dsub_rn(1.0, __dmul_rn(s, s)));
}

// floor of 0 <= x < 2^32 without a cvt instruction: round-down add of 2^52, low word.
__device__ __forceinline__ unsigned lya_floor_u32(double x)
{
    return (unsigned)__double2loint(__dadd_rd(x, 4503599627370496.0));
}

// Per-forest-pair constants for binning pixel pairs.
struct PairBin {
    double c, s;        // cos, sin of theta/2
    double cx, sy;      // pow2 path: c*inv_par, s*inv_perp (exact scalings)
};

// Bin of a pixel pair, -1 outside the grid.  POW2: bin widths are powers of two, so
// (|d|*c)*inv == |d|*(c*inv) exactly and r < r_max <=> floor(r*inv) < n.
template <bool POW2>
__device__ __forceinline__ int lya_pix_bin(const BinParams &bp, const PairBin &g, double chi_i, double chi_j)
{
    double d = __dsub_rn(chi_i, chi_j);
    double t = __dadd_rn(chi_i, chi_j);
    if (POW2) {
        unsigned bx = lya_floor_u32(__dmul_rn(fabs(d), g.cx));
        unsigned by = lya_floor_u32(__dmul_rn(t, g.sy));
        bool ok = (bx < (unsigned)bp.n_par) & (by < (unsigned)bp.n_perp);
        return ok ? (int)(bx * (unsigned)bp.n_perp + by) : -1;
    } else {
        double rpar = __dmul_rn(fabs(d), g.c);
        double rperp = __dmul_rn(t, g.s);
        bool ok = (rpar < bp.rpar_max) & (rperp < bp.rperp_max);
        unsigned bx = min(lya_floor_u32(__dmul_rn(rpar, bp.inv_par)), (unsigned)(bp.n_par - 1));
        unsigned by = min(lya_floor_u32(__dmul_rn(rperp, bp.inv_perp)), (unsigned)(bp.n_perp - 1));
        return ok ? (int)(bx * (unsigned)bp.n_perp + by) : -1;
    }
}

// Same bin test, TRANSPOSED index b_perp * n_par + b_par (the internal order of the D accumulator:
// the bins a forest pair touches are then contiguous runs of b_par inside <= 6 columns).
template <bool POW2>
__device__ __forceinline__ int lya_pix_bin_t(const BinParams &bp, const PairBin &g, double chi_i, double chi_j)
{
    double d = __dsub_rn(chi_i, chi_j);
    double t = __dadd_rn(chi_i, chi_j);
    unsigned bx, by;
    bool ok;
    if (POW2) {
        bx = lya_floor_u32(__dmul_rn(fabs(d), g.cx));
        by = lya_floor_u32(__dmul_rn(t, g.sy));
        ok = (bx < (unsigned)bp.n_par) & (by < (unsigned)bp.n_perp);
    } else {
        double rpar = __dmul_rn(fabs(d), g.c);
        double rperp = __dmul_rn(t, g.s);
        ok = (rpar < bp.rpar_max) & (rperp < bp.rperp_max);
        bx = min(lya_floor_u32(__dmul_rn(rpar, bp.inv_par)), (unsigned)(bp.n_par - 1));
        by = min(lya_floor_u32(__dmul_rn(rperp, bp.inv_perp)), (unsigned)(bp.n_perp - 1));
    }
    return ok ? (int)(by * (unsigned)bp.n_par + bx) : -1;
}
// API bin index (b_par * n_perp + b_perp) -> transposed
__device__ __forceinline__ int lya_bin_tr(const BinParams &bp, int A)
{
    const int bx = A / bp.n_perp;
    return (A - bx * bp.n_perp) * bp.n_par + bx;
}

__device__ __forceinline__ PairBin lya_make_pairbin(const BinParams &bp, double s, double c)
{
    PairBin g;
    g.c = c; g.s = s;
    g.cx = __dmul_rn(c, bp.inv_par);
    g.sy = __dmul_rn(s, bp.inv_perp);
    return g;
}

// r_perp column of a pixel pair with chi_i + chi_j = t, or n_perp when r_perp >= rperp_max
// (same operations as lya_pix_bin, so the value is the column lya_pix_bin assigns).
template <bool POW2>
__device__ __forceinline__ int lya_col_of(const BinParams &bp, const PairBin &g, double t)
{
    if (POW2) {
        unsigned by = lya_floor_u32(__dmul_rn(t, g.sy));
        return (by < (unsigned)bp.n_perp) ? (int)by : bp.n_perp;
    } else {
        double rperp = __dmul_rn(t, g.s);
        if (!(rperp < bp.rperp_max)) return bp.n_perp;
        return (int)min(lya_floor_u32(__dmul_rn(rperp, bp.inv_perp)), (unsigned)(bp.n_perp - 1));
    }
}

// Diagonal stride of a forest pair: the smallest ds with ds * (smallest pixel spacing of q) > r_par bin width
// (margin 1e-6).  Lanes of one row step that sit ds pixels of q apart then hold pairs in different r_par bins on
// each side of chi_i = chi_j.  Returns a large number for a single-pixel q.
__device__ __forceinline__ int lya_pair_stride(const BinParams &bp, const PairBin &g, const ForestHead &hq)
{
    const double x = __dmul_rn(__dmul_rn(hq.dmin, g.c), bp.inv_par);     // spacing in bin widths
    if (x > 1.000001) return 1;
    if (!(x > 1.000001 / 64.0)) return 64;
    return (int)(1.000001 / x) + 1;
}

// Which kernel takes this forest pair?  (warp-uniform; identical in the bucketing pass and in the kernels.)
// c_first: column of the pair's first pixels.  Returns the bucket key (see LyaBuckets).
template <bool POW2>
__device__ __forceinline__ int lya_pair_key(const BinParams &bp, const PairBin &g, const ForestHead &hp,
                                            const ForestHead &hq, int &c_first)
{
    c_first = bp.n_perp;
    if (hp.len == 0 || hq.len == 0) return LYA_KEY_SKIP(bp.n_perp);
    c_first = lya_col_of<POW2>(bp, g, __dadd_rn(hp.chi0, hq.chi0));
    if (c_first >= bp.n_perp) return LYA_KEY_SKIP(bp.n_perp);       // r_perp grows with both pixels
    int c_last = lya_col_of<POW2>(bp, g, __dadd_rn(hp.chi1, hq.chi1));
    if (c_last >= bp.n_perp) c_last = bp.n_perp - 1;
    if (c_last - c_first >= LYA_NCOL) return LYA_KEY_GENERIC(bp.n_perp);
    const int len = max(hp.len, hq.len);
    const int ds = lya_pair_stride(bp, g, hq);
    if (len <= LYA_FAST_TILE && ds == 1) return c_first;
    if (len <= LYA_FAST_TILE2 && ds <= LYA_DS_MAX) return bp.n_perp + c_first;
    if (len <= LYA_LONG_TILE && ds <= LYA_DS_MAX_LONG) return LYA_KEY_LONG(bp.n_perp);
    return LYA_KEY_GENERIC(bp.n_perp);
}
#endif
