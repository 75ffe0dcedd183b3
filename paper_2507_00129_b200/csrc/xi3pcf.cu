// xi3pcf.cu -- NEXT-4 (lya_xi3pcf): brute-force anisotropic three-point correlation function, eq. 2.8
// (triangle variables of PAPER.md:108, Fig. 2, Fig. 5):
//
//   xi3_A = sum_A (d_i w_i)(d_j w_j)(d_k w_k) / sum_A w_i w_j w_k     over pixels i, j, k of three DISTINCT forests
//
// Readings T1-T7 of DESIGN.md (the paper fixes neither the vertex convention nor the line of sight nor the
// flattening): every ORDERED triple (i; j, k) counts, i the main vertex; X = chi u; d1 = X_j - X_i,
// d2 = X_k - X_i; a side takes part iff 0 < r < r_max; line of sight = the vertex forest's unit vector;
// cos theta = (d . u_i) / r; cos alpha = (d1 . d2) / (r1 r2); b_r = (int)(r n_r / r_max); b_theta = number of
// table edges C_m = cos(m pi / n_theta) with cos theta <= C_m (the table is an input); b_alpha =
// (int)((cos alpha + 1) n_cosa / 2) clamped; A = (((b_r1 n_r + b_r2) n_cosa + b_alpha) n_theta + b_theta1) n_theta + b_theta2.
// Every operation is one separately rounded binary64 operation (explicit _rn intrinsics), so the triplet
// counts are bit-identical to the CPU oracle's.
//
// Design: "we stick to the brute-force algorithm".  The forest-pair list (any superset of the
// pairs with two pixels closer than r_max, e.g. lya_neighbours with rperp_max = r_max: r_perp <= the 3-D
// separation) is turned into an adjacency list in both directions.  One CTA per main-vertex forest p; for each
// of its pixels i the CTA gathers the pixels of p's neighbours that lie inside the sphere of radius r_max
// (side vector, length, bins, weights) into shared memory, then its threads run over the UNORDERED pairs {j, k} of
// that list (the two orders of the sides share cos alpha bit for bit and land in mirrored bins: the second order
// is added by k_xi3_finalize), with three reductions per unordered pair into the L2-resident accumulators
// (20 x 20 x 20 x 10 x 10 bins x 24 B = 19 MB).
#include <math.h>
#include <stdlib.h>
#include "lya_internal.cuh"

namespace {

constexpr int T3_THREADS = 512;
constexpr int T3_CAP = 2048;                 // pixels inside the sphere of one main-vertex pixel (shared-memory list)

struct Tri3Params {
    lya_forests f;
    double r_max, inv_r, nhalf;
    int n_r, n_theta, n_cosa;
    const double *cosedge;                   // [n_theta - 1]
    const unsigned long long *adj_off;       // [n_forest + 1]
    const int32_t *adj;                      // neighbours of every forest (both directions)
    double *S3, *W3;                         // HALF accumulators: one entry per unordered {j, k} (see k_xi3)
    unsigned long long *N3;
    unsigned long long *counters;            // [0] triples binned, [3] error (capacity)
};

__global__ void k_adj_count(const int32_t *pq, int64_t n, int64_t n_forest, unsigned *deg, unsigned long long *err)
{
    const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int p = pq[2 * k], q = pq[2 * k + 1];
    if ((unsigned)p >= (unsigned)n_forest || (unsigned)q >= (unsigned)n_forest) { atomicMax(err, (unsigned long long)LYA_DEV_BAD_PAIR); return; }
    atomicAdd(&deg[p], 1u);
    atomicAdd(&deg[q], 1u);
}
__global__ void k_adj_fill(const int32_t *pq, int64_t n, int64_t n_forest, const unsigned long long *off, unsigned *cursor, int32_t *adj)
{
    const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int p = pq[2 * k], q = pq[2 * k + 1];
    if ((unsigned)p >= (unsigned)n_forest || (unsigned)q >= (unsigned)n_forest) return;
    adj[off[p] + atomicAdd(&cursor[p], 1u)] = q;
    adj[off[q] + atomicAdd(&cursor[q], 1u)] = p;
}

struct Tri3Smem {
    double2 xy[T3_CAP], zr[T3_CAP], aw[T3_CAP];   // side vector (dx, dy), (dz, r), (a = w delta, w): three 16-byte reads per pixel
    int2 bf[T3_CAP];                              // (b_r | b_theta << 8, forest)
    unsigned n;
};

// The two orders (i; j, k) and (i; k, j) of a triple share every rounded operation of cos alpha (products and
// r1 r2 commute, the additions keep their order), so they fall in the bins A(b_r1, b_r2, b_a, b_t1, b_t2) and
// swap(A) = A(b_r2, b_r1, b_a, b_t2, b_t1) with the same weights up to the rounding order of T7.  The kernel therefore
// walks every UNORDERED {j, k} once and adds it to A only; k_xi3_finalize returns acc[A] + acc[swap(A)] (half the
// geometry, half the reductions; the counts stay exact, S3 and W3 move by an ulp per term).
__global__ void __launch_bounds__(T3_THREADS) k_xi3(Tri3Params P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Tri3Smem &sm = *(Tri3Smem *)smem_raw;
    const int p = blockIdx.x;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, n_warps = T3_THREADS / 32;
    const int64_t op = P.f.pix_off[p];
    const int np = (int)(P.f.pix_off[p + 1] - op);
    const unsigned long long a0 = P.adj_off[p], a1 = P.adj_off[p + 1];
    if (np == 0 || a1 - a0 < 2) return;                        // a triangle needs two other forests
    const double ux = P.f.ux[p], uy = P.f.uy[p], uz = P.f.uz[p];
    unsigned long long n_tri = 0;
    for (int ii = 0; ii < np; ++ii) {
        const double ci = P.f.chi[op + ii], wi = P.f.w[op + ii], ai = wi * P.f.delta[op + ii];
        const double xi0 = __dmul_rn(ci, ux), xi1 = __dmul_rn(ci, uy), xi2 = __dmul_rn(ci, uz);      // T1
        __syncthreads();
        if (threadIdx.x == 0) sm.n = 0u;
        __syncthreads();
        // ---- gather: warps over the neighbour forests, lanes over their pixels (T3, T4, T5 per side).  A pixel
        //      with |chi_j - chi_i| beyond r_max (plus a margin for |u| = 1 +- 1e-9) cannot be inside the sphere ----
        const double guard = P.r_max * (1.0 + 1e-6) + 1e-6;
        for (unsigned long long e = a0 + wid; e < a1; e += n_warps) {
            const int q = P.adj[e];
            const int64_t oq = P.f.pix_off[q];
            const int nq = (int)(P.f.pix_off[q + 1] - oq);
            const double qx = P.f.ux[q], qy = P.f.uy[q], qz = P.f.uz[q];
            for (int j = lane; j < nq; j += 32) {
                const double cj = P.f.chi[oq + j];
                if (fabs(cj - ci) > guard + 4e-9 * (cj + ci)) continue;
                const double d0 = __dsub_rn(__dmul_rn(cj, qx), xi0), d1 = __dsub_rn(__dmul_rn(cj, qy), xi1), d2 = __dsub_rn(__dmul_rn(cj, qz), xi2);
                const double r = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(d0, d0), __dmul_rn(d1, d1)), __dmul_rn(d2, d2)));
                if (r > 0.0 && r < P.r_max) {
                    int br = __double2int_rz(__dmul_rn(r, P.inv_r));
                    if (br > P.n_r - 1) br = P.n_r - 1;
                    const double ct = __ddiv_rn(__dadd_rn(__dadd_rn(__dmul_rn(d0, ux), __dmul_rn(d1, uy)), __dmul_rn(d2, uz)), r);
                    int bt = 0;
                    for (int m = 0; m < P.n_theta - 1; ++m) bt += (ct <= P.cosedge[m]) ? 1 : 0;
                    const unsigned s = atomicAdd(&sm.n, 1u);
                    if (s < (unsigned)T3_CAP) {
                        const double wj = P.f.w[oq + j];
                        sm.xy[s] = make_double2(d0, d1); sm.zr[s] = make_double2(d2, r);
                        sm.aw[s] = make_double2(wj * P.f.delta[oq + j], wj);
                        sm.bf[s] = make_int2(br | (bt << 8), q);
                    }
                }
            }
        }
        __syncthreads();
        const unsigned C = sm.n;
        if (C > (unsigned)T3_CAP) {                            // (CTA-uniform) more pixels in the sphere than the list holds
            if (threadIdx.x == 0) atomicMax(&P.counters[3], (unsigned long long)LYA_DEV_TOO_LONG);
            return;
        }
        if (C < 2u) continue;
        // ---- unordered pairs {j, k} of gathered pixels from two different forests (T2, T4-T7): k = j + d (mod C)
        //      for the offsets d = 1 .. (C - 1) / 2 and every j, plus d = C / 2 for j < C / 2 when C is even; the
        //      threads run over the flat index d * C + j, so a warp reads neighbouring list entries ----
        const unsigned half = (C - 1u) >> 1;
        const unsigned total = C * half + ((C & 1u) ? 0u : (C >> 1));
        const unsigned qd = (unsigned)T3_THREADS / C, rd = (unsigned)T3_THREADS % C;
        unsigned d = 1u + threadIdx.x / C, j = threadIdx.x % C;
        for (unsigned t = threadIdx.x; t < total; t += T3_THREADS) {
            unsigned k = j + d;
            if (k >= C) k -= C;
            const int2 bj = sm.bf[j], bk = sm.bf[k];
            if (bj.y != bk.y) {
                const double2 xy1 = sm.xy[j], zr1 = sm.zr[j], aw1 = sm.aw[j];
                const double2 xy2 = sm.xy[k], zr2 = sm.zr[k], aw2 = sm.aw[k];
                const double dot = __dadd_rn(__dadd_rn(__dmul_rn(xy1.x, xy2.x), __dmul_rn(xy1.y, xy2.y)), __dmul_rn(zr1.x, zr2.x));
                const double ca = __ddiv_rn(dot, __dmul_rn(zr1.y, zr2.y));
                int ba = __double2int_rz(__dmul_rn(__dadd_rn(ca, 1.0), P.nhalf));
                ba = max(0, min(ba, P.n_cosa - 1));
                const unsigned A = (unsigned)(((((bj.x & 0xff) * P.n_r + (bk.x & 0xff)) * P.n_cosa + ba) * P.n_theta + (bj.x >> 8)) * P.n_theta + (bk.x >> 8));
                atomicAdd(&P.S3[A], (ai * aw1.x) * aw2.x);     // (three RED.E.ADD: the kernel runs at the rate at which L2 takes
                atomicAdd(&P.W3[A], (wi * aw1.y) * aw2.y);     //  scattered 8-byte reductions, 2.0e11 / s -- profiles/r2l_xi3pcf.md)
                atomicAdd(&P.N3[A], 1ull);
                n_tri += 2;
            }
            j += rd; d += qd;
            if (j >= C) { j -= C; ++d; }
        }
    }
    // ordered triples counted by this CTA
    for (int o = 16; o > 0; o >>= 1) n_tri += __shfl_xor_sync(0xffffffffu, n_tri, o);
    if (lane == 0 && n_tri) atomicAdd(&P.counters[0], n_tri);
}

// result[A] = acc[A] + acc[swap(A)] (both orders of the two sides, see k_xi3), xi3 = S3 / W3
__global__ void k_xi3_finalize(const double *S, const double *W, const unsigned long long *N, int64_t nb, int n_r, int n_cosa, int n_theta,
                               double *S_out, double *W_out, unsigned long long *N_out, double *xi_out)
{
    const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (k >= nb) return;
    int64_t v = k;
    const int t2 = (int)(v % n_theta); v /= n_theta;
    const int t1 = (int)(v % n_theta); v /= n_theta;
    const int ba = (int)(v % n_cosa); v /= n_cosa;
    const int b2 = (int)(v % n_r), b1 = (int)(v / n_r);
    const int64_t ks = ((((int64_t)b2 * n_r + b1) * n_cosa + ba) * n_theta + t2) * n_theta + t1;
    const double s = S[k] + S[ks], w = W[k] + W[ks];
    const unsigned long long n = N[k] + N[ks];
    if (S_out) S_out[k] = s;
    if (W_out) W_out[k] = w;
    if (N_out) N_out[k] = n;
    if (xi_out) xi_out[k] = (w != 0.0) ? s / w : 0.0;
}

}  // namespace

extern "C" int64_t lya_tri_nbins(const lya_tri_binning *tb)
{
    if (!tb || tb->n_r < 1 || tb->n_theta < 1 || tb->n_cosa < 1) return 0;
    return (int64_t)tb->n_r * tb->n_r * tb->n_cosa * tb->n_theta * tb->n_theta;
}

extern "C" lya_status lya_xi3pcf(lya_ctx *ctx, const lya_forests *f, const lya_tri_binning *tb, const double *cos_theta_edges,
                                 const lya_pairs *pairs, double *S3, double *W3, uint64_t *N3, double *xi3, lya_stats *stats)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    if (!tb || !pairs) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi3pcf: NULL argument");
    if (!(tb->r_max > 0) || !isfinite(tb->r_max) || tb->n_r < 1 || tb->n_theta < 1 || tb->n_cosa < 1)
        return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi3pcf: need r_max > 0 and n_r, n_theta, n_cosa >= 1");
    if (tb->n_r > 255 || tb->n_theta > 255 || tb->r_max > 1e5 || lya_tri_nbins(tb) > ((int64_t)1 << 24))
        return lya_fail(ctx, LYA_ERR_CAPACITY, "lya_xi3pcf: at most 255 bins per variable, 2^24 triangle bins, r_max <= 1e5");
    if (tb->n_theta > 1 && !cos_theta_edges) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi3pcf: cos_theta_edges is NULL");
    lya_status st = lya_check_forests_host(ctx, f, true, true, false);
    if (st) return st;
    if (f->n_forest > 0 && !(f->ux && f->uy && f->uz)) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi3pcf needs ux,uy,uz (device)");
    LYA_CUDA(lya_enter(ctx));
    st = lya_validate_forests(ctx, f, true, false, NULL);
    if (st) return st;
    const int64_t nb = lya_tri_nbins(tb), nf = f->n_forest, n = pairs->n;
    cudaStream_t s = ctx->stream;
    double *acc = NULL;
    unsigned *deg = NULL, *cursor = NULL;
    unsigned long long *off = NULL, *tmp = NULL;
    int32_t *adj = NULL;
    auto cleanup = [&]() { lya_free(acc); lya_free(deg); lya_free(cursor); lya_free(off); lya_free(tmp); lya_free(adj); };
    cudaError_t e = lya_malloc(&acc, sizeof(double) * 3 * (size_t)nb);
    if (e == cudaSuccess) e = lya_malloc(&deg, sizeof(unsigned) * (size_t)(nf + 1));
    if (e == cudaSuccess) e = lya_malloc(&cursor, sizeof(unsigned) * (size_t)(nf + 1));
    if (e == cudaSuccess) e = lya_malloc(&off, sizeof(unsigned long long) * (size_t)(nf + 2));
    if (e == cudaSuccess) e = lya_malloc(&tmp, sizeof(unsigned long long) * (size_t)(nf / 2048 + 4));
    if (e == cudaSuccess) e = lya_malloc(&adj, sizeof(int32_t) * (size_t)(2 * n + 1));
    if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "lya_malloc(lya_xi3pcf)"); }
    cudaEventRecord(ctx->ev[3], s);
    cudaMemsetAsync(acc, 0, sizeof(double) * 3 * (size_t)nb, s);
    cudaMemsetAsync(deg, 0, sizeof(unsigned) * (size_t)(nf + 1), s);
    cudaMemsetAsync(cursor, 0, sizeof(unsigned) * (size_t)(nf + 1), s);
    cudaMemsetAsync(ctx->d_counters, 0, 8 * sizeof(unsigned long long), s);
    if (n > 0) { k_adj_count<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(pairs->pq, n, nf, deg, ctx->d_counters + 3); lya_note_launch(); }
    unsigned long long h[4] = {0, 0, 0, 0};
    if (nf > 0) {
        e = lya_exclusive_scan(deg, off, nf, tmp, s);
        if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "lya_xi3pcf (adjacency scan)"); }
        if (n > 0) { k_adj_fill<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(pairs->pq, n, nf, off, cursor, adj); lya_note_launch(); }
        Tri3Params P;
        P.f = *f; P.r_max = tb->r_max; P.inv_r = (double)tb->n_r / tb->r_max; P.nhalf = (double)tb->n_cosa / 2.0;
        P.n_r = tb->n_r; P.n_theta = tb->n_theta; P.n_cosa = tb->n_cosa;
        P.cosedge = cos_theta_edges; P.adj_off = off; P.adj = adj;
        P.S3 = acc; P.W3 = acc + nb; P.N3 = (unsigned long long *)(acc + 2 * nb);
        P.counters = ctx->d_counters;
        const size_t smem = sizeof(Tri3Smem);
        e = cudaFuncSetAttribute(k_xi3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        cudaEventRecord(ctx->ev[0], s);
        if (e == cudaSuccess) { k_xi3<<<(unsigned)nf, T3_THREADS, smem, s>>>(P); lya_note_launch(); }
        cudaEventRecord(ctx->ev[1], s);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "k_xi3 launch"); }
    } else {
        cudaEventRecord(ctx->ev[0], s);
        cudaEventRecord(ctx->ev[1], s);
    }
    { k_xi3_finalize<<<(unsigned)((nb + 255) / 256), 256, 0, s>>>(acc, acc + nb, (unsigned long long *)(acc + 2 * nb), nb, tb->n_r, tb->n_cosa, tb->n_theta, S3, W3, (unsigned long long *)N3, xi3); lya_note_launch(); }
    cudaEventRecord(ctx->ev[2], s);
    e = cudaMemcpyAsync(h, ctx->d_counters, sizeof(h), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cleanup();
    if (e != cudaSuccess) return lya_cuda_fail(ctx, e, "lya_xi3pcf");
    if (h[3] == LYA_DEV_BAD_PAIR) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "pair list refers to a forest outside [0, n_forest)");
    if (h[3] == LYA_DEV_TOO_LONG) return lya_fail(ctx, LYA_ERR_CAPACITY, "lya_xi3pcf: more than %d pixels within r_max of one pixel", T3_CAP);
    if (stats) {
        memset(stats, 0, sizeof(*stats));
        stats->n_forest_pairs = (uint64_t)n;
        stats->n_binned = h[0];
        stats->n_evaluated = h[0];
        cudaEventElapsedTime(&stats->ms_main, ctx->ev[0], ctx->ev[1]);
        cudaEventElapsedTime(&stats->ms_total, ctx->ev[3], ctx->ev[2]);
    }
    return LYA_OK;
}
