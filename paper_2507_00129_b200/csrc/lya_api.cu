// lya_api.cu -- context, argument validation, pair-list handles and the host-buffer
// end-to-end entry point of liblya.so (include/lya.h).
#include <math.h>
#include <stdarg.h>
#include <stdlib.h>
#include "lya_internal.cuh"

unsigned long long g_lya_launches = 0;
thread_local cudaStream_t tl_lya_stream = 0;
thread_local bool tl_lya_pool = false;

cudaError_t lya_enter(lya_ctx *ctx)
{
    cudaError_t e = cudaSetDevice(ctx->device);
    tl_lya_stream = ctx->stream;
    tl_lya_pool = ctx->use_pool != 0;
    return e;
}
extern "C" uint64_t lya_launch_count(void) { return g_lya_launches; }

extern "C" const char *lya_version(void) { return "lya-b200 0.1 (sm_100a)"; }

lya_status lya_fail(lya_ctx *ctx, lya_status st, const char *fmt, ...)
{
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
        va_end(ap);
    }
    return st;
}

lya_status lya_cuda_fail(lya_ctx *ctx, cudaError_t e, const char *what)
{
    lya_status st = (e == cudaErrorMemoryAllocation) ? LYA_ERR_OOM : LYA_ERR_CUDA;
    return lya_fail(ctx, st, "CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
}

extern "C" lya_status lya_create(lya_ctx **out, int device, void *cuda_stream)
{
    if (!out) return LYA_ERR_INVALID_ARG;
    *out = NULL;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev <= 0 || device < 0 || device >= n_dev)
        return LYA_ERR_CUDA;   // no CPU fallback: the library needs a CUDA device
    lya_ctx *ctx = (lya_ctx *)calloc(1, sizeof(lya_ctx));
    if (!ctx) return LYA_ERR_OOM;
    ctx->device = device;
    ctx->stream = (cudaStream_t)cuda_stream;
    if (cudaSetDevice(device) != cudaSuccess) { free(ctx); return LYA_ERR_CUDA; }
    {   // stream-ordered scratch allocation with a pool that keeps freed blocks (see lya_internal.cuh)
        int has_pools = 0;
        cudaMemPool_t pool;
        if (cudaDeviceGetAttribute(&has_pools, cudaDevAttrMemoryPoolsSupported, device) == cudaSuccess && has_pools &&
            cudaDeviceGetDefaultMemPool(&pool, device) == cudaSuccess) {
            unsigned long long keep = ~0ull;
            ctx->use_pool = cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep) == cudaSuccess;
        }
        cudaGetLastError();
        tl_lya_stream = ctx->stream;
        tl_lya_pool = ctx->use_pool != 0;
    }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { free(ctx); return LYA_ERR_CUDA; }
    ctx->sm_count = prop.multiProcessorCount;
    if (cudaMalloc(&ctx->d_counters, 16 * sizeof(unsigned long long)) != cudaSuccess) { free(ctx); return LYA_ERR_OOM; }
    for (int i = 0; i < 4; ++i)
        if (cudaEventCreate(&ctx->ev[i]) != cudaSuccess) { cudaFree(ctx->d_counters); free(ctx); return LYA_ERR_CUDA; }
    ctx->force_generic = 0;
    ctx->generic_diagonals = 2;
    ctx->check_holders = 0;
    ctx->xi_merge_every = 1ull << 31;
    ctx->err[0] = 0;
    *out = ctx;
    return LYA_OK;
}

extern "C" void lya_destroy(lya_ctx *ctx)
{
    if (!ctx) return;
    lya_enter(ctx);
    for (int i = 0; i < 4; ++i) cudaEventDestroy(ctx->ev[i]);
    cudaFree(ctx->d_counters);
    if (ctx->use_pool) {                              // hand the cached scratch back to the driver
        cudaMemPool_t pool;
        cudaStreamSynchronize(ctx->stream);
        if (cudaDeviceGetDefaultMemPool(&pool, ctx->device) == cudaSuccess) cudaMemPoolTrimTo(pool, 0);
    }
    free(ctx);
}

extern "C" const char *lya_last_error(const lya_ctx *ctx) { return ctx ? ctx->err : "null ctx"; }

extern "C" lya_status lya_set_option(lya_ctx *ctx, lya_option opt, int64_t value)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    switch (opt) {
    case LYA_OPT_FORCE_GENERIC:
        if (value != 0 && value != 1) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "LYA_OPT_FORCE_GENERIC takes 0 or 1");
        ctx->force_generic = (int)value;
        return LYA_OK;
    case LYA_OPT_GENERIC_DIAGONALS:
        if (value != 1 && value != 2 && value != 4) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "LYA_OPT_GENERIC_DIAGONALS takes 1, 2 or 4");
        ctx->generic_diagonals = (int)value;
        return LYA_OK;
    case LYA_OPT_XI_MERGE_EVERY:
        if (value < 1 || value > ((int64_t)1 << 31)) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "LYA_OPT_XI_MERGE_EVERY takes 1 .. 2^31");
        ctx->xi_merge_every = (unsigned long long)value;
        return LYA_OK;
    case LYA_OPT_CHECK_HOLDERS:
        if (value != 0 && value != 1) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "LYA_OPT_CHECK_HOLDERS takes 0 or 1");
        ctx->check_holders = (int)value;
        return LYA_OK;
    default:
        return lya_fail(ctx, LYA_ERR_INVALID_ARG, "unknown option %d", (int)opt);
    }
}

lya_status lya_check_binning(lya_ctx *ctx, const lya_binning *b)
{
    if (!b) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "binning is NULL");
    if (!(b->rpar_max > 0) || !(b->rperp_max > 0) || !isfinite(b->rpar_max) || !isfinite(b->rperp_max) ||
        b->n_par < 1 || b->n_perp < 1)
        return lya_fail(ctx, LYA_ERR_INVALID_ARG, "binning: need r*_max > 0 and n_* >= 1");
    if ((int64_t)b->n_par * b->n_perp > LYA_MAX_BINS)
        return lya_fail(ctx, LYA_ERR_CAPACITY, "binning: n_par*n_perp = %lld exceeds %d",
                        (long long)b->n_par * b->n_perp, LYA_MAX_BINS);
    if (b->rpar_max / b->n_par < 0.01 || b->rperp_max / b->n_perp < 0.01)
        return lya_fail(ctx, LYA_ERR_CAPACITY, "binning: bin width below 0.01");
    // padding / sentinel pixels sit at chi = 1e7 and 2e7 and must stay far outside any grid
    if (b->rpar_max > 1e5 || b->rperp_max > 1e5)
        return lya_fail(ctx, LYA_ERR_CAPACITY, "binning: r*_max above 1e5");
    return LYA_OK;
}

lya_status lya_check_forests_host(lya_ctx *ctx, const lya_forests *f, bool need_u, bool need_delta, bool need_loglam)
{
    if (!f) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "forests is NULL");
    if (f->n_forest < 0 || f->n_pix < 0) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "negative sizes");
    if (f->n_forest >= ((int64_t)1 << 31) || f->n_pix >= ((int64_t)1 << 40))
        return lya_fail(ctx, LYA_ERR_CAPACITY, "n_forest must be < 2^31 and n_pix < 2^40");
    if (!f->pix_off) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "pix_off is NULL");
    if (f->n_pix > 0 && (!f->chi || !f->w)) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "chi / w is NULL");
    if (need_delta && f->n_pix > 0 && !f->delta) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "delta is NULL");
    if (need_loglam && f->n_pix > 0 && !f->loglam) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "loglam is NULL");
    if (need_u && f->n_forest > 0) {
        bool have_u = f->ux && f->uy && f->uz;
        bool have_radec = f->ra && f->dec;
        if (!have_u && !have_radec)
            return lya_fail(ctx, LYA_ERR_INVALID_ARG, "need ux,uy,uz (all three) or ra,dec");
        if (!have_u && (f->ux || f->uy || f->uz))
            return lya_fail(ctx, LYA_ERR_INVALID_ARG, "ux,uy,uz must be given together");
    }
    return LYA_OK;
}

// ---- device validation ---------------------------------------------------------
__global__ void k_validate(lya_forests f, bool need_delta, bool need_loglam, unsigned *d_err, int *d_maxlen)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= f.n_forest) return;
    int64_t a = f.pix_off[p], b = f.pix_off[p + 1];
    unsigned err = 0;
    if (p == 0 && a != 0) err = LYA_DEV_BAD_OFFSETS;
    if (p == f.n_forest - 1 && b != f.n_pix) err = LYA_DEV_BAD_OFFSETS;
    if (a > b || a < 0 || b > f.n_pix) { atomicMax(d_err, (unsigned)LYA_DEV_BAD_OFFSETS); return; }
    if (b - a > (1 << 20)) { atomicMax(d_err, (unsigned)LYA_DEV_TOO_LONG); return; }
    double prev = -1.0;
    for (int64_t k = a; k < b; ++k) {
        double c = f.chi[k], w = f.w[k];
        bool fin = isfinite(c) && isfinite(w) && (c >= 0.0) && (c < LYA_CHI_MAX) && (w >= 0.0);
        if (need_delta) fin = fin && isfinite(f.delta[k]);
        if (need_loglam) fin = fin && isfinite(f.loglam[k]);
        if (!fin) err = max(err, (unsigned)LYA_DEV_NONFINITE);
        else if (!(c > prev)) err = max(err, (unsigned)LYA_DEV_UNSORTED);
        prev = c;
    }
    if (f.ux) {
        const double n2 = f.ux[p] * f.ux[p] + f.uy[p] * f.uy[p] + f.uz[p] * f.uz[p];
        if (!(isfinite(n2) && fabs(n2 - 1.0) <= 1e-9)) err = max(err, (unsigned)LYA_DEV_NONFINITE);   // finite and of unit length
    } else if (f.ra) {
        if (!(isfinite(f.ra[p]) && isfinite(f.dec[p]))) err = max(err, (unsigned)LYA_DEV_NONFINITE);
    }
    if (err) atomicMax(d_err, err);
    atomicMax(d_maxlen, (int)(b - a));
}

lya_status lya_validate_forests(lya_ctx *ctx, const lya_forests *f, bool need_delta, bool need_loglam, int *max_len)
{
    if (max_len) *max_len = 0;
    if (f->n_forest == 0) {
        return LYA_OK;
    }
    unsigned *d_err = (unsigned *)(ctx->d_counters + 8);
    int *d_maxlen = (int *)(ctx->d_counters + 9);
    LYA_CUDA(cudaMemsetAsync(ctx->d_counters + 8, 0, 2 * sizeof(unsigned long long), ctx->stream));
    int threads = 128;
    int64_t blocks = (f->n_forest + threads - 1) / threads;
    { k_validate<<<(unsigned)blocks, threads, 0, ctx->stream>>>(*f, need_delta, need_loglam, d_err, d_maxlen); lya_note_launch(); }
    LYA_CUDA(cudaGetLastError());
    unsigned long long h[2];
    LYA_CUDA(cudaMemcpyAsync(h, ctx->d_counters + 8, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
    LYA_CUDA(cudaStreamSynchronize(ctx->stream));
    unsigned err = (unsigned)h[0];
    if (max_len) *max_len = (int)h[1];
    switch (err) {
    case LYA_DEV_OK: return LYA_OK;
    case LYA_DEV_BAD_OFFSETS: return lya_fail(ctx, LYA_ERR_INVALID_ARG, "pix_off must start at 0, be non-decreasing and end at n_pix");
    case LYA_DEV_NONFINITE: return lya_fail(ctx, LYA_ERR_INVALID_ARG, "non-finite input, w < 0, chi outside [0, 1e6), or a sightline vector that is not of unit length (1e-9)");
    case LYA_DEV_UNSORTED: return lya_fail(ctx, LYA_ERR_UNSORTED, "chi is not strictly increasing inside a forest");
    case LYA_DEV_TOO_LONG: return lya_fail(ctx, LYA_ERR_CAPACITY, "a forest has more than 2^20 pixels");
    default: return lya_fail(ctx, LYA_ERR_INVALID_ARG, "catalogue validation failed (%u)", err);
    }
}

// ---- pair-list handles ------------------------------------------------------------
__global__ void k_import_pairs(const int32_t *in, int32_t *out, int64_t n, unsigned *d_err)
{
    int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (k >= n) return;
    int32_t p = in[2 * k], q = in[2 * k + 1];
    if (p == q || p < 0 || q < 0) atomicMax(d_err, (unsigned)LYA_DEV_BAD_PAIR);
    out[2 * k] = min(p, q);
    out[2 * k + 1] = max(p, q);
}

extern "C" lya_status lya_pairs_import(lya_ctx *ctx, const int32_t *pq, int64_t n_pairs, lya_pairs **out)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    if (!out || n_pairs < 0 || (n_pairs > 0 && !pq)) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_pairs_import: bad arguments");
    *out = NULL;
    LYA_CUDA(lya_enter(ctx));
    lya_pairs *pl = (lya_pairs *)calloc(1, sizeof(lya_pairs));
    if (!pl) return lya_fail(ctx, LYA_ERR_OOM, "host allocation failed");
    pl->n = n_pairs;
    if (n_pairs > 0) {
        cudaError_t e = lya_malloc(&pl->pq, sizeof(int32_t) * 2 * (size_t)n_pairs);
        if (e != cudaSuccess) { free(pl); return lya_cuda_fail(ctx, e, "lya_malloc(pair list)"); }
        unsigned *d_err = (unsigned *)(ctx->d_counters + 8);
        cudaMemsetAsync(d_err, 0, sizeof(unsigned long long), ctx->stream);
        int threads = 256;
        { k_import_pairs<<<(unsigned)((n_pairs + threads - 1) / threads), threads, 0, ctx->stream>>>(pq, pl->pq, n_pairs, d_err); lya_note_launch(); }
        unsigned long long h = 0;
        e = cudaMemcpyAsync(&h, d_err, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) { lya_free(pl->pq); free(pl); return lya_cuda_fail(ctx, e, "lya_pairs_import"); }
        if ((unsigned)h != 0) { lya_free(pl->pq); free(pl); return lya_fail(ctx, LYA_ERR_INVALID_ARG, "pair list has p == q or a negative index"); }
    }
    *out = pl;
    return LYA_OK;
}

extern "C" lya_status lya_pairs_export(lya_ctx *ctx, const lya_pairs *pairs, int32_t *pq)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    if (!pairs || (pairs->n > 0 && !pq)) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_pairs_export: bad arguments");
    LYA_CUDA(lya_enter(ctx));
    if (pairs->n > 0)
        LYA_CUDA(cudaMemcpyAsync(pq, pairs->pq, sizeof(int32_t) * 2 * (size_t)pairs->n, cudaMemcpyDeviceToDevice, ctx->stream));
    return LYA_OK;
}

extern "C" int64_t lya_pairs_count(const lya_pairs *pairs) { return pairs ? pairs->n : 0; }

extern "C" void lya_pairs_free(lya_ctx *ctx, lya_pairs *pairs)
{
    if (!pairs) return;
    if (ctx) lya_enter(ctx);
    if (pairs->pq) lya_free(pairs->pq);
    free(pairs);
}

// ---- end-to-end with host buffers ----------------------------------------------------
namespace {
struct DevBuf {
    void *p = nullptr;
    ~DevBuf() { if (p) lya_free(p); }
    cudaError_t alloc(size_t bytes) { return lya_malloc(&p, bytes ? bytes : 1); }
};
}

extern "C" lya_status lya_run_host(lya_ctx *ctx, const lya_forests *fh, const lya_binning *b,
                                   int do_xi, int do_dmat, double reject_fraction, uint64_t seed,
                                   double *S, double *W, uint64_t *N, double *xi, double *D, double *Wd,
                                   int64_t *n_pairs_out, lya_stats *stats_xi, lya_stats *stats_dmat)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    lya_status st = lya_check_binning(ctx, b);
    if (st) return st;
    st = lya_check_forests_host(ctx, fh, true, do_xi != 0, do_dmat != 0);
    if (st) return st;
    if (!(fh->ux && fh->uy && fh->uz)) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_run_host needs ux,uy,uz");
    LYA_CUDA(lya_enter(ctx));
    const int64_t nf = fh->n_forest, np = fh->n_pix;
    const int64_t nb = (int64_t)b->n_par * b->n_perp;
    DevBuf ux, uy, uz, off, chi, w, delta, loglam, dS, dW, dN, dxi, dD, dWd;
    LYA_CUDA(ux.alloc(8 * nf)); LYA_CUDA(uy.alloc(8 * nf)); LYA_CUDA(uz.alloc(8 * nf));
    LYA_CUDA(off.alloc(8 * (nf + 1))); LYA_CUDA(chi.alloc(8 * np)); LYA_CUDA(w.alloc(8 * np));
    if (do_xi) LYA_CUDA(delta.alloc(8 * np));
    if (do_dmat) LYA_CUDA(loglam.alloc(8 * np));
    cudaStream_t s = ctx->stream;
    LYA_CUDA(cudaMemcpyAsync(ux.p, fh->ux, 8 * nf, cudaMemcpyHostToDevice, s));
    LYA_CUDA(cudaMemcpyAsync(uy.p, fh->uy, 8 * nf, cudaMemcpyHostToDevice, s));
    LYA_CUDA(cudaMemcpyAsync(uz.p, fh->uz, 8 * nf, cudaMemcpyHostToDevice, s));
    LYA_CUDA(cudaMemcpyAsync(off.p, fh->pix_off, 8 * (nf + 1), cudaMemcpyHostToDevice, s));
    LYA_CUDA(cudaMemcpyAsync(chi.p, fh->chi, 8 * np, cudaMemcpyHostToDevice, s));
    LYA_CUDA(cudaMemcpyAsync(w.p, fh->w, 8 * np, cudaMemcpyHostToDevice, s));
    if (do_xi) LYA_CUDA(cudaMemcpyAsync(delta.p, fh->delta, 8 * np, cudaMemcpyHostToDevice, s));
    if (do_dmat) LYA_CUDA(cudaMemcpyAsync(loglam.p, fh->loglam, 8 * np, cudaMemcpyHostToDevice, s));
    lya_forests fd;
    memset(&fd, 0, sizeof(fd));
    fd.n_forest = nf; fd.n_pix = np;
    fd.ux = (double *)ux.p; fd.uy = (double *)uy.p; fd.uz = (double *)uz.p;
    fd.pix_off = (int64_t *)off.p; fd.chi = (double *)chi.p; fd.w = (double *)w.p;
    fd.delta = do_xi ? (double *)delta.p : NULL; fd.loglam = do_dmat ? (double *)loglam.p : NULL;

    lya_pairs *pairs = NULL;
    int64_t n_pairs = 0;
    st = lya_neighbours(ctx, &fd, b, &pairs, &n_pairs);
    if (st) return st;
    if (n_pairs_out) *n_pairs_out = n_pairs;
    lya_plan *plan = NULL;
    st = lya_plan_create(ctx, &fd, b, pairs, do_xi != 0, do_dmat != 0, &plan);
    lya_pairs_free(ctx, pairs);                       // (the plan holds its own bucket-sorted copy)
    pairs = NULL;
    if (st) return st;
    if (do_xi) {
        cudaError_t e = dS.alloc(8 * nb);
        if (e == cudaSuccess) e = dW.alloc(8 * nb);
        if (e == cudaSuccess) e = dN.alloc(8 * nb);
        if (e == cudaSuccess) e = dxi.alloc(8 * nb);
        if (e != cudaSuccess) { lya_plan_free(ctx, plan); return lya_cuda_fail(ctx, e, "lya_malloc(xi outputs)"); }
        st = lya_xi2pcf_plan(ctx, plan, (double *)dS.p, (double *)dW.p, (uint64_t *)dN.p, (double *)dxi.p, stats_xi);
        if (st) { lya_plan_free(ctx, plan); return st; }
        if (S) cudaMemcpyAsync(S, dS.p, 8 * nb, cudaMemcpyDeviceToHost, s);
        if (W) cudaMemcpyAsync(W, dW.p, 8 * nb, cudaMemcpyDeviceToHost, s);
        if (N) cudaMemcpyAsync(N, dN.p, 8 * nb, cudaMemcpyDeviceToHost, s);
        if (xi) cudaMemcpyAsync(xi, dxi.p, 8 * nb, cudaMemcpyDeviceToHost, s);
    }
    if (do_dmat) {
        cudaError_t e = dD.alloc(8 * nb * nb);
        if (e == cudaSuccess) e = dWd.alloc(8 * nb);
        if (e != cudaSuccess) { lya_plan_free(ctx, plan); return lya_cuda_fail(ctx, e, "lya_malloc(D outputs)"); }
        st = lya_dmat_plan(ctx, plan, reject_fraction, seed, (double *)dD.p, NULL, (double *)dWd.p, stats_dmat);
        if (st) { lya_plan_free(ctx, plan); return st; }
        if (D) cudaMemcpyAsync(D, dD.p, 8 * nb * nb, cudaMemcpyDeviceToHost, s);
        if (Wd) cudaMemcpyAsync(Wd, dWd.p, 8 * nb, cudaMemcpyDeviceToHost, s);
    }
    cudaError_t e = cudaStreamSynchronize(s);
    lya_plan_free(ctx, plan);

    if (e != cudaSuccess) return lya_cuda_fail(ctx, e, "lya_run_host");
    return LYA_OK;
}
