// prep.cu -- per-call preparation shared by the pair kernels (lya_xi2pcf, lya_dmat):
//
//  (1) lya_prep_build: a padded, 16-byte aligned SoA copy of the catalogue (so a warp can
//      stage a forest with 16-byte vector loads) with the per-pixel products the kernels
//      need -- w*delta for eq. 2.4, and u = L - Lbar, w/sum w, w u/sum w u^2 for eq. 2.7
//       -- plus one 80-byte head per forest (unit vector, first/last chi,
//      smallest chi spacing, packed offset, length).
//  (2) lya_bucket_pairs: a stable counting sort of the forest-pair list by the r_perp
//      column of the pair's first pixel pair.  Pairs of one bucket touch the same
//      <= LYA_NCOL bin columns, which lets every warp keep a private (n_par x LYA_NCOL)
//      sub-histogram in shared memory across many forest pairs.
#include <stdlib.h>
#include "lya_internal.cuh"

namespace {

// ---- (1) prepared catalogue ---------------------------------------------------------
__global__ void k_pad_len(const int64_t *pix_off, int64_t n_forest, unsigned *padlen)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= n_forest) return;
    int64_t n = pix_off[p + 1] - pix_off[p];
    padlen[p] = (unsigned)((n + 1) & ~(int64_t)1);
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_min(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// one warp per forest
template <bool XI, bool DMAT>
__global__ void k_pack(lya_forests f, const unsigned long long *off2, LyaPrep P)
{
    const int64_t p = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (p >= f.n_forest) return;
    const int64_t a = f.pix_off[p];
    const int n = (int)(f.pix_off[p + 1] - a);
    const long long o = (long long)off2[p];
    const int npad = (n + 1) & ~1;
    // Lbar = L_0 + sum w (L - L_0) / sum w: the differences are exact, so Lbar is the correctly rounded mean but
    // for rare ties.  (sum w L / sum w in plain fp64 can be an ulp off, and for a forest whose L spans 1e-4 an ulp
    // of Lbar is 1e-11 of u = L - Lbar: visible in D where eta should cancel exactly, e.g. a 2-pixel forest.)
    double dmin = 1e300, sw = 0.0, swl = 0.0;
    const double l0 = (DMAT && n > 0) ? f.loglam[a] : 0.0;
    for (int t = lane; t < n; t += 32) {
        double c = f.chi[a + t];
        if (t + 1 < n) dmin = fmin(dmin, f.chi[a + t + 1] - c);
        if (DMAT) { double w = f.w[a + t]; sw += w; swl += w * (f.loglam[a + t] - l0); }
    }
    dmin = warp_min(dmin);
    double lbar = 0.0, invS = 0.0, invV = 0.0;
    int flags = 0;
    if (DMAT) {
        sw = warp_sum(sw); swl = warp_sum(swl);
        lbar = (sw > 0.0) ? l0 + swl / sw : 0.0;
        double v = 0.0;
        for (int t = lane; t < n; t += 32) { double u = f.loglam[a + t] - lbar; v += f.w[a + t] * u * u; }
        v = warp_sum(v);
        // degenerate (reading R-7): no weight, or all weighted L equal up to rounding of L - Lbar
        const double tiny = 1e-12 * fabs(lbar);
        const bool ok = (sw > 0.0) && (v > sw * tiny * tiny);
        invS = ok ? 1.0 / sw : 0.0;
        invV = ok ? 1.0 / v : 0.0;
        flags = ok ? 0 : 1;
    }
    for (int t = lane; t < npad; t += 32) {
        const bool in = t < n;
        const double c = in ? f.chi[a + t] : LYA_CHI_SENTINEL;
        const double w = in ? f.w[a + t] : 0.0;
        P.w[o + t] = w;
        if (XI) { P.chi[o + t] = c; P.a[o + t] = in ? w * f.delta[a + t] : 0.0; }
        if (DMAT) {
            const double u = in ? f.loglam[a + t] - lbar : 0.0;
            P.u[o + t] = u;
            P.ce[o + t] = make_double2(c, w * invS);
            P.eg[o + t] = w * u * invV;
        }
    }
    if (lane == 0) {
        ForestHead h;
        h.ux = f.ux[p]; h.uy = f.uy[p]; h.uz = f.uz[p];
        h.dmin = dmin;
        h.chi0 = n ? f.chi[a] : 0.0;
        h.chi1 = n ? f.chi[a + n - 1] : 0.0;
        h.off = o; h.pix0 = (long long)a; h.len = n; h.flags = flags;
        P.head[p] = h;
    }
}

// ---- (2) bucketing ------------------------------------------------------------------
constexpr int BK_TILE = 2048;            // pairs per tile (one warp walks a tile in order)
constexpr int BK_MAX_KEYS = 64 * 4 + 3;  // LYA_N_KEYS(n_perp) <= this

template <bool POW2>
__device__ __forceinline__ int pair_key(const ForestHead *head, int64_t n_forest, const BinParams &bp, int p, int q,
                                        unsigned long long &visited, int &bad)
{
    if ((unsigned)p >= (unsigned)n_forest || (unsigned)q >= (unsigned)n_forest) { bad = max(bad, (int)LYA_DEV_BAD_PAIR); return LYA_KEY_SKIP(bp.n_perp); }
    const ForestHead hp = head[p], hq = head[q];
    if ((hp.flags | hq.flags) & 1) bad = max(bad, (int)LYA_DEV_DEGENERATE);   // (only set by a dmat catalogue)
    visited += (unsigned long long)hp.len * (unsigned long long)hq.len;
    double s, c;
    lya_pair_sc(hp.ux, hp.uy, hp.uz, hq.ux, hq.uy, hq.uz, s, c);
    const PairBin g = lya_make_pairbin(bp, s, c);
    int c_first;
    return lya_pair_key<POW2>(bp, g, hp, hq, c_first);
}

// counts[key * n_tiles + tile]; one warp per tile.  force_generic: every in-grid pair gets
// key n_perp (the grid has too many r_par rows for a sub-histogram).
template <bool POW2>
__global__ void k_bucket_count(const ForestHead *head, int64_t n_forest, BinParams bp, const int32_t *pq, int64_t n,
                               int64_t n_tiles, int force_generic, unsigned char *keys, unsigned *counts,
                               unsigned long long *counters)
{
    __shared__ unsigned hist[4][BK_MAX_KEYS];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t tile = blockIdx.x * (int64_t)(blockDim.x >> 5) + w;
    const int nk = LYA_N_KEYS(bp.n_perp);
    for (int k = lane; k < nk; k += 32) hist[w][k] = 0;
    __syncwarp();
    unsigned long long visited = 0;
    int bad = 0;
    if (tile < n_tiles) {
        const int64_t k0 = tile * BK_TILE, k1 = min(k0 + BK_TILE, n);
        for (int64_t k = k0 + lane; k < k1; k += 32) {
            const int2 e = ((const int2 *)pq)[k];
            int key = pair_key<POW2>(head, n_forest, bp, e.x, e.y, visited, bad);
            if (force_generic && key < LYA_KEY_GENERIC(bp.n_perp)) key = LYA_KEY_GENERIC(bp.n_perp);
            keys[k] = (unsigned char)min(key, 255);
            atomicAdd(&hist[w][key], 1u);
        }
        __syncwarp();
        for (int k = lane; k < nk; k += 32) counts[(int64_t)k * n_tiles + tile] = hist[w][k];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) visited += __shfl_xor_sync(0xffffffffu, visited, o);
    bad = __reduce_max_sync(0xffffffffu, bad);
    if (lane == 0) {
        if (visited) atomicAdd(&counters[1], visited);
        if (bad) atomicMax(&counters[3], (unsigned long long)bad);
    }
}

// stable scatter: one warp per tile walks it in order, 32 pairs at a time
__global__ void k_bucket_scatter(const int32_t *pq, const unsigned char *keys, int64_t n, int64_t n_tiles, int nk,
                                 const unsigned long long *offsets, int32_t *out)
{
    __shared__ unsigned long long cur[4][BK_MAX_KEYS];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t tile = blockIdx.x * (int64_t)(blockDim.x >> 5) + w;
    if (tile >= n_tiles) return;
    for (int k = lane; k < nk; k += 32) cur[w][k] = offsets[(int64_t)k * n_tiles + tile];
    __syncwarp();
    const int64_t k0 = tile * BK_TILE, k1 = min(k0 + BK_TILE, n);
    for (int64_t kb = k0; kb < k1; kb += 32) {
        const int64_t k = kb + lane;
        const bool in = k < k1;
        const int key = in ? (int)keys[k] : -1;
        const unsigned peers = __match_any_sync(0xffffffffu, key);
        const int rank = __popc(peers & ((1u << lane) - 1u));
        if (in) {
            const unsigned long long pos = cur[w][key] + rank;
            ((int2 *)out)[pos] = ((const int2 *)pq)[k];
        }
        __syncwarp();
        if (in && rank == 0) cur[w][key] += __popc(peers);      // one leader per key
        __syncwarp();
    }
}

}  // namespace

void lya_prep_free(LyaPrep *p)
{
    if (p && p->base) { lya_free(p->base); p->base = NULL; }
}

lya_status lya_prep_build(lya_ctx *ctx, const lya_forests *f, bool want_xi, bool want_dmat, LyaPrep *out)
{
    memset(out, 0, sizeof(*out));
    const int64_t n = f->n_forest;
    out->n_forest = n;
    if (n == 0) return LYA_OK;
    cudaStream_t s = ctx->stream;
    unsigned *padlen = NULL;
    unsigned long long *off2 = NULL, *tmp = NULL;
    LYA_CUDA(lya_malloc(&padlen, sizeof(unsigned) * (size_t)n));
    cudaError_t e = lya_malloc(&off2, sizeof(unsigned long long) * (size_t)(n + 1));
    if (e == cudaSuccess) e = lya_malloc(&tmp, sizeof(unsigned long long) * (size_t)(n / 2048 + 4));
    if (e != cudaSuccess) { lya_free(padlen); lya_free(off2); return lya_cuda_fail(ctx, e, "lya_malloc(prep scratch)"); }
    auto drop = [&]() { lya_free(padlen); lya_free(off2); lya_free(tmp); };
    { k_pad_len<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(f->pix_off, n, padlen); lya_note_launch(); }
    e = lya_exclusive_scan(padlen, off2, n, tmp, s);
    unsigned long long total = 0;
    if (e == cudaSuccess) e = cudaMemcpyAsync(&total, off2 + n, sizeof(total), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { drop(); return lya_cuda_fail(ctx, e, "prep scan"); }
    out->n_pack = (int64_t)total;
    const int n_arr = 1 + (want_xi ? 2 : 0) + (want_dmat ? 4 : 0);
    const size_t head_bytes = sizeof(ForestHead) * (size_t)n;
    const size_t arr_bytes = ((size_t)total * 8 + 255) & ~(size_t)255;
    e = lya_malloc(&out->base, head_bytes + arr_bytes * n_arr + 256);
    if (e != cudaSuccess) { drop(); out->base = NULL; return lya_cuda_fail(ctx, e, "lya_malloc(prepared catalogue)"); }
    char *b = (char *)out->base;
    out->head = (ForestHead *)b; b += (head_bytes + 255) & ~(size_t)255;
    out->w = (double *)b; b += arr_bytes;
    if (want_xi) { out->chi = (double *)b; b += arr_bytes; out->a = (double *)b; b += arr_bytes; }
    if (want_dmat) { out->ce = (double2 *)b; b += 2 * arr_bytes; out->eg = (double *)b; b += arr_bytes; out->u = (double *)b; b += arr_bytes; }
    const unsigned blocks = (unsigned)((n * 32 + 255) / 256);
    if (want_xi && want_dmat) { k_pack<true, true><<<blocks, 256, 0, s>>>(*f, off2, *out); lya_note_launch(); }
    else if (want_xi) { k_pack<true, false><<<blocks, 256, 0, s>>>(*f, off2, *out); lya_note_launch(); }
    else if (want_dmat) { k_pack<false, true><<<blocks, 256, 0, s>>>(*f, off2, *out); lya_note_launch(); }
    else { k_pack<false, false><<<blocks, 256, 0, s>>>(*f, off2, *out); lya_note_launch(); }
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);      // scratch is freed below
    drop();
    if (e != cudaSuccess) { lya_prep_free(out); return lya_cuda_fail(ctx, e, "k_pack"); }
    return LYA_OK;
}

void lya_buckets_free(LyaBuckets *b)
{
    if (b && b->pq) { lya_free(b->pq); b->pq = NULL; }
}

// counters[1] += visited, counters[3] = error flag (the caller zeroes ctx->d_counters first)
lya_status lya_bucket_pairs(lya_ctx *ctx, const LyaPrep *prep, const BinParams *bp, const lya_pairs *pairs,
                            int force_generic, LyaBuckets *out)
{
    memset(out, 0, sizeof(*out));
    const int64_t n = pairs->n;
    out->n = n;
    if (n == 0) return LYA_OK;
    const int nk = LYA_N_KEYS(bp->n_perp);
    if (nk > BK_MAX_KEYS || nk > 256) return lya_fail(ctx, LYA_ERR_CAPACITY, "n_perp above %d", 126);
    cudaStream_t s = ctx->stream;
    const int64_t n_tiles = (n + BK_TILE - 1) / BK_TILE;
    const int64_t n_cnt = n_tiles * nk;
    unsigned char *keys = NULL;
    unsigned *counts = NULL;
    unsigned long long *offsets = NULL, *tmp = NULL;
    cudaError_t e = lya_malloc(&keys, (size_t)n);
    if (e == cudaSuccess) e = lya_malloc(&counts, sizeof(unsigned) * (size_t)n_cnt);
    if (e == cudaSuccess) e = lya_malloc(&offsets, sizeof(unsigned long long) * (size_t)(n_cnt + 1));
    if (e == cudaSuccess) e = lya_malloc(&tmp, sizeof(unsigned long long) * (size_t)(n_cnt / 2048 + 4));
    if (e == cudaSuccess) e = lya_malloc(&out->pq, sizeof(int32_t) * 2 * (size_t)n);
    auto drop = [&]() { lya_free(keys); lya_free(counts); lya_free(offsets); lya_free(tmp); };
    if (e != cudaSuccess) { drop(); lya_free(out->pq); out->pq = NULL; return lya_cuda_fail(ctx, e, "lya_malloc(bucketing)"); }
    const unsigned blocks = (unsigned)((n_tiles + 3) / 4);
    if (bp->pow2)
        { k_bucket_count<true><<<blocks, 128, 0, s>>>(prep->head, prep->n_forest, *bp, pairs->pq, n, n_tiles, force_generic, keys, counts, ctx->d_counters); lya_note_launch(); }
    else
        { k_bucket_count<false><<<blocks, 128, 0, s>>>(prep->head, prep->n_forest, *bp, pairs->pq, n, n_tiles, force_generic, keys, counts, ctx->d_counters); lya_note_launch(); }
    e = lya_exclusive_scan(counts, offsets, n_cnt, tmp, s);
    if (e == cudaSuccess) {
        { k_bucket_scatter<<<blocks, 128, 0, s>>>(pairs->pq, keys, n, n_tiles, nk, offsets, out->pq); lya_note_launch(); }
        e = cudaGetLastError();
    }
    unsigned long long h_start[4] = {0, 0, 0, 0};     // start of class 1, of the long range, of the generic range, of the skipped pairs
    unsigned long long h_cnt[4];
    const int first_key[4] = {bp->n_perp, LYA_KEY_LONG(bp->n_perp), LYA_KEY_GENERIC(bp->n_perp), LYA_KEY_SKIP(bp->n_perp)};
    for (int k = 0; k < 4 && e == cudaSuccess; ++k)
        e = cudaMemcpyAsync(&h_start[k], offsets + (int64_t)first_key[k] * n_tiles, 8, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h_cnt, ctx->d_counters, sizeof(h_cnt), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    drop();
    if (e != cudaSuccess) { lya_buckets_free(out); return lya_cuda_fail(ctx, e, "pair bucketing"); }
    out->n_fast = (int64_t)h_start[0];
    out->n_fast2 = (int64_t)(h_start[1] - h_start[0]);
    out->n_long = (int64_t)(h_start[2] - h_start[1]);
    out->n_generic = (int64_t)(h_start[3] - h_start[2]);
    out->n_skip = n - (int64_t)h_start[3];
    out->visited = h_cnt[1];
    out->bad_pair = (int)h_cnt[3];
    return LYA_OK;
}

// ---- plans ---------------------------------------------------------------------------------------
extern "C" void lya_plan_free(lya_ctx *ctx, lya_plan *pl)
{
    if (!pl) return;
    if (ctx) lya_enter(ctx);
    lya_prep_free(&pl->prep);
    lya_buckets_free(&pl->bk);
    if (pl->pq) lya_free(pl->pq);
    free(pl);
}

extern "C" lya_status lya_plan_create(lya_ctx *ctx, const lya_forests *f, const lya_binning *b, const lya_pairs *pairs,
                                      int want_xi, int want_dmat, lya_plan **out)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    if (!out) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_plan_create: out is NULL");
    *out = NULL;
    if (!pairs) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_plan_create: pairs is NULL");
    if (!want_xi && !want_dmat) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_plan_create: want_xi or want_dmat");
    lya_status st = lya_check_binning(ctx, b);
    if (st) return st;
    st = lya_check_forests_host(ctx, f, true, want_xi != 0, want_dmat != 0);
    if (st) return st;
    if (f->n_forest > 0 && !(f->ux && f->uy && f->uz))
        return lya_fail(ctx, LYA_ERR_INVALID_ARG, "the pair kernels need ux,uy,uz (device); derive them once with the catalogue");
    LYA_CUDA(lya_enter(ctx));
    int max_len = 0;
    st = lya_validate_forests(ctx, f, want_xi != 0, want_dmat != 0, &max_len);
    if (st) return st;
    lya_plan *pl = (lya_plan *)calloc(1, sizeof(lya_plan));
    if (!pl) return lya_fail(ctx, LYA_ERR_OOM, "host allocation failed");
    pl->f = *f; pl->b = *b; pl->bp = lya_make_binparams(b);
    pl->has_xi = want_xi != 0; pl->has_dmat = want_dmat != 0;
    pl->n_pairs = pairs->n; pl->max_len = max_len;
    pl->use_fast = pairs->n > 0 && b->n_par <= LYA_FAST_NPAR_MAX && LYA_N_KEYS(b->n_perp) <= 256 && !ctx->force_generic;
    cudaStream_t s = ctx->stream;
    if (pl->use_fast) {
        st = lya_prep_build(ctx, f, pl->has_xi, pl->has_dmat, &pl->prep);
        if (st) { lya_plan_free(ctx, pl); return st; }
        cudaMemsetAsync(ctx->d_counters, 0, 8 * sizeof(unsigned long long), s);
        st = lya_bucket_pairs(ctx, &pl->prep, &pl->bp, pairs, 0, &pl->bk);
        if (st) { lya_plan_free(ctx, pl); return st; }
        if (pl->bk.bad_pair == LYA_DEV_BAD_PAIR) {
            lya_plan_free(ctx, pl);
            return lya_fail(ctx, LYA_ERR_INVALID_ARG, "pair list refers to a forest outside [0, n_forest)");
        }
        pl->listed_degenerate = pl->bk.bad_pair == LYA_DEV_DEGENERATE;
        pl->visited = pl->bk.visited;
    } else if (pairs->n > 0) {
        cudaError_t e = lya_malloc(&pl->pq, sizeof(int32_t) * 2 * (size_t)pairs->n);
        if (e == cudaSuccess) e = cudaMemcpyAsync(pl->pq, pairs->pq, sizeof(int32_t) * 2 * (size_t)pairs->n, cudaMemcpyDeviceToDevice, s);
        if (e != cudaSuccess) { lya_plan_free(ctx, pl); return lya_cuda_fail(ctx, e, "lya_plan_create (pair list copy)"); }
    }
    *out = pl;
    return LYA_OK;
}
