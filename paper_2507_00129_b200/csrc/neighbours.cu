// neighbours.cu -- stage 1 (lya_neighbours): on-device neighbour search.
//
// PAPER.md:79 / :124: "our algorithm only takes forests within a pre-ordered
// neighborhood defined by this maximum distance" (HEALPix in the paper).  Here: a
// uniform 3-D cell grid over the unit vectors.  A listed pair satisfies
//     (chi_p[0] + chi_q[0]) * s < rperp_max          (reading G4, s = chord/2)
// so its chord is below 2*s_max with s_max = rperp_max / (2 * min_p chi_p[0]); with a
// cell edge >= that chord every listed pair lives in adjacent cells (27-cell search).
// A 3-D grid has no RA wrap or pole special cases (pin P9).
//
// Pipeline: prep (unit vectors, chi_min) -> cell histogram -> exclusive scan ->
// scatter -> per-cell sort by forest id (deterministic order) -> count (warp per
// forest) -> exclusive scan -> fill.  Output: int32 [n_pairs][2], p < q, grouped by p
// in cell order (spatially coherent, which the pair kernels rely on for L2 reuse).
#include <math.h>
#include <stdlib.h>
#include "lya_internal.cuh"

namespace {

constexpr int G_MAX = 128;          // cells per axis (dense G^3 table, <= 2M cells)
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;       // per thread -> 2048 per block

// ---- exclusive scan: in (u32) -> out (u64), out[n] = total ------------------------
__global__ void k_scan_block(const unsigned *in, unsigned long long *out, unsigned long long *block_sums, int64_t n)
{
    __shared__ unsigned long long warp_tot[SCAN_THREADS / 32];
    int64_t base = (int64_t)blockIdx.x * (SCAN_THREADS * SCAN_ITEMS) + (int64_t)threadIdx.x * SCAN_ITEMS;
    unsigned long long v[SCAN_ITEMS], sum = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        v[k] = (base + k < n) ? in[base + k] : 0;
        sum += v[k];
    }
    unsigned long long incl = sum;
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned long long t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) warp_tot[wid] = incl;
    __syncthreads();
    unsigned long long woff = 0;
    for (int k = 0; k < wid; ++k) woff += warp_tot[k];
    unsigned long long run = woff + incl - sum;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < n) out[base + k] = run;
        run += v[k];
    }
    if (threadIdx.x == SCAN_THREADS - 1) block_sums[blockIdx.x] = woff + incl;
}

__global__ void k_scan_sums(unsigned long long *block_sums, int64_t nblocks, unsigned long long *total)
{
    // single thread block, sequential over chunks (nblocks <= a few thousand)
    __shared__ unsigned long long carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int64_t base = 0; base < nblocks; base += blockDim.x) {
        int64_t i = base + threadIdx.x;
        unsigned long long v = (i < nblocks) ? block_sums[i] : 0, incl = v;
        int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
        __shared__ unsigned long long wt[32];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            unsigned long long t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) wt[wid] = incl;
        __syncthreads();
        unsigned long long woff = 0;
        for (int k = 0; k < wid; ++k) woff += wt[k];
        unsigned long long c = carry;
        if (i < nblocks) block_sums[i] = c + woff + incl - v;
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry = c + woff + incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) *total = carry;
}

__global__ void k_scan_add(unsigned long long *out, const unsigned long long *block_sums, int64_t n,
                           const unsigned long long *total)
{
    int64_t i = (int64_t)blockIdx.x * (SCAN_THREADS * SCAN_ITEMS) + threadIdx.x;
    unsigned long long add = block_sums[blockIdx.x];
    for (int k = 0; k < SCAN_ITEMS; ++k, i += SCAN_THREADS)
        if (i < n) out[i] += add;
    if (blockIdx.x == 0 && threadIdx.x == 0) out[n] = *total;
}

// out must hold n+1 entries; tmp must hold ceil(n/2048)+1 entries.
cudaError_t exclusive_scan(const unsigned *in, unsigned long long *out, int64_t n, unsigned long long *tmp, cudaStream_t s)
{
    int64_t nblocks = (n + SCAN_THREADS * SCAN_ITEMS - 1) / (SCAN_THREADS * SCAN_ITEMS);
    if (nblocks == 0) {
        return cudaMemsetAsync(out, 0, sizeof(unsigned long long), s);
    }
    { k_scan_block<<<(unsigned)nblocks, SCAN_THREADS, 0, s>>>(in, out, tmp, n); lya_note_launch(); }
    { k_scan_sums<<<1, 1024, 0, s>>>(tmp, nblocks, tmp + nblocks); lya_note_launch(); }
    { k_scan_add<<<(unsigned)nblocks, SCAN_THREADS, 0, s>>>(out, tmp, n, tmp + nblocks); lya_note_launch(); }
    return cudaGetLastError();
}

// ---- prep --------------------------------------------------------------------------
struct SortedForests {
    double *ux, *uy, *uz, *chimin;   // in cell order
    int *id;                         // original forest index
};

__global__ void k_prep(lya_forests f, double *ux, double *uy, double *uz, double *chimin,
                       unsigned long long *d_min_bits)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= f.n_forest) return;
    double x, y, z;
    if (f.ux) { x = f.ux[p]; y = f.uy[p]; z = f.uz[p]; }
    else {
        double sd, cd, sr, cr;
        sincos(f.dec[p], &sd, &cd);
        sincos(f.ra[p], &sr, &cr);
        x = cd * cr; y = cd * sr; z = sd;
    }
    ux[p] = x; uy[p] = y; uz[p] = z;
    int64_t a = f.pix_off[p], b = f.pix_off[p + 1];
    double cm = (b > a) ? f.chi[a] : -1.0;      // -1: empty forest, never listed
    chimin[p] = cm;
    if (b > a) atomicMin(d_min_bits, (unsigned long long)__double_as_longlong(cm));   // chi >= 0: bit order == value order
}

__device__ __forceinline__ int cell_coord(double u, int G)
{
    int c = (int)((u + 1.0) * (0.5 * G));
    return min(max(c, 0), G - 1);
}

__global__ void k_cell_hist(const double *ux, const double *uy, const double *uz, const double *chimin,
                            int64_t n, int G, int *cell_of, unsigned *hist)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= n) return;
    int c = -1;
    if (chimin[p] >= 0.0) {
        c = (cell_coord(uz[p], G) * G + cell_coord(uy[p], G)) * G + cell_coord(ux[p], G);
        atomicAdd(&hist[c], 1u);
    }
    cell_of[p] = c;
}

__global__ void k_cell_scatter(const int *cell_of, int64_t n, const unsigned long long *cell_start,
                               unsigned *cursor, int *sorted_id)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= n) return;
    int c = cell_of[p];
    if (c < 0) return;
    unsigned slot = atomicAdd(&cursor[c], 1u);
    sorted_id[cell_start[c] + slot] = (int)p;
}

// deterministic order inside a cell: sort by forest id (insertion sort for the usual small cells, an in-place
// heap sort for crowded ones, e.g. a whole catalogue in one cell when the admissible chord exceeds the sphere)
__global__ void k_cell_sort(const unsigned long long *cell_start, int64_t n_cells, int *sorted_id)
{
    int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (c >= n_cells) return;
    const int64_t a = cell_start[c], n = (int64_t)cell_start[c + 1] - a;
    if (n < 2) return;
    int *v = sorted_id + a;
    if (n <= 64) {
        for (int64_t i = 1; i < n; ++i) {
            const int x = v[i];
            int64_t j = i - 1;
            while (j >= 0 && v[j] > x) { v[j + 1] = v[j]; --j; }
            v[j + 1] = x;
        }
        return;
    }
    auto sift = [&](int64_t root, int64_t end) {            // max-heap on v[0, end)
        for (;;) {
            int64_t child = 2 * root + 1;
            if (child >= end) break;
            if (child + 1 < end && v[child + 1] > v[child]) ++child;
            if (v[root] >= v[child]) break;
            const int t = v[root]; v[root] = v[child]; v[child] = t;
            root = child;
        }
    };
    for (int64_t i = n / 2 - 1; i >= 0; --i) sift(i, n);
    for (int64_t end = n - 1; end > 0; --end) {
        const int t = v[0]; v[0] = v[end]; v[end] = t;
        sift(0, end);
    }
}

__global__ void k_gather_sorted(const int *sorted_id, int64_t m, const double *ux, const double *uy, const double *uz,
                                const double *chimin, SortedForests sf)
{
    int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (k >= m) return;
    int p = sorted_id[k];
    sf.ux[k] = ux[p]; sf.uy[k] = uy[p]; sf.uz[k] = uz[p]; sf.chimin[k] = chimin[p]; sf.id[k] = p;
}

// ---- count / fill: one warp per forest (in cell order) --------------------------------
// FILL = false: counts[k] = number of partners b with id_b > id_a that pass G4.
// FILL = true : writes them at pq[offsets[k] ...] in (cell, position) order.
template <bool FILL>
__global__ void k_pairs(SortedForests sf, int64_t m, const unsigned long long *cell_start, int G, double rperp_max,
                        unsigned *counts, const unsigned long long *offsets, int32_t *pq)
{
    int64_t k = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (k >= m) return;
    double ax = sf.ux[k], ay = sf.uy[k], az = sf.uz[k], acm = sf.chimin[k];
    int aid = sf.id[k];
    int cx = cell_coord(ax, G), cy = cell_coord(ay, G), cz = cell_coord(az, G);
    unsigned long long out = FILL ? offsets[k] : 0;
    unsigned total = 0;
    for (int dz = -1; dz <= 1; ++dz) {
        int z = cz + dz;
        if (z < 0 || z >= G) continue;
        for (int dy = -1; dy <= 1; ++dy) {
            int y = cy + dy;
            if (y < 0 || y >= G) continue;
            // the three x-cells are contiguous in the table: one candidate range
            int x0 = max(cx - 1, 0), x1 = min(cx + 1, G - 1);
            int64_t c0 = ((int64_t)z * G + y) * G + x0, c1 = ((int64_t)z * G + y) * G + x1;
            int64_t beg = cell_start[c0], end = cell_start[c1 + 1];
            for (int64_t t = beg; t < end; t += 32) {
                int64_t j = t + lane;
                bool hit = false;
                int bid = 0;
                if (j < end) {
                    bid = sf.id[j];
                    if (bid > aid) {
                        double s, c;
                        lya_pair_sc(ax, ay, az, sf.ux[j], sf.uy[j], sf.uz[j], s, c);
                        // G4: (chi_min_p + chi_min_q) * s < rperp_max  (+ is commutative: order-free)
                        hit = __dmul_rn(__dadd_rn(acm, sf.chimin[j]), s) < rperp_max;
                    }
                }
                unsigned bal = __ballot_sync(0xffffffffu, hit);
                if (FILL && hit) {
                    unsigned long long pos = out + __popc(bal & ((1u << lane) - 1u));
                    pq[2 * pos] = aid;
                    pq[2 * pos + 1] = bid;
                }
                int n = __popc(bal);
                out += n;
                total += n;
            }
        }
    }
    if (!FILL && lane == 0) counts[k] = total;
}

struct Scratch {
    void *ptrs[24];
    int n = 0;
    ~Scratch() { for (int i = 0; i < n; ++i) lya_free(ptrs[i]); }
    template <class T> cudaError_t alloc(T **p, size_t count)
    {
        cudaError_t e = lya_malloc(p, sizeof(T) * (count ? count : 1));
        if (e == cudaSuccess) ptrs[n++] = *p;
        return e;
    }
};

}  // namespace

cudaError_t lya_exclusive_scan(const unsigned *in, unsigned long long *out, int64_t n, unsigned long long *tmp,
                               cudaStream_t s)
{
    return exclusive_scan(in, out, n, tmp, s);
}

extern "C" lya_status lya_neighbours(lya_ctx *ctx, const lya_forests *f, const lya_binning *b,
                                     lya_pairs **out, int64_t *n_pairs)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    if (!out || !n_pairs) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_neighbours: out / n_pairs is NULL");
    *out = NULL; *n_pairs = 0;
    lya_status st = lya_check_binning(ctx, b);
    if (st) return st;
    st = lya_check_forests_host(ctx, f, true, false, false);
    if (st) return st;
    LYA_CUDA(lya_enter(ctx));
    st = lya_validate_forests(ctx, f, false, false, NULL);
    if (st) return st;

    lya_pairs *pl = (lya_pairs *)calloc(1, sizeof(lya_pairs));
    if (!pl) return lya_fail(ctx, LYA_ERR_OOM, "host allocation failed");
    const int64_t n = f->n_forest;
    if (n < 2) { *out = pl; return LYA_OK; }

    cudaStream_t s = ctx->stream;
    Scratch sc;
    double *ux, *uy, *uz, *chimin;
    int *cell_of, *sorted_id;
    unsigned *counts;
    unsigned long long *offsets, *scan_tmp;
    SortedForests sf;
#define NB_ALLOC(ptr, cnt) do { cudaError_t e_ = sc.alloc(&(ptr), (size_t)(cnt)); if (e_ != cudaSuccess) { free(pl); return lya_cuda_fail(ctx, e_, "lya_malloc(neighbour scratch)"); } } while (0)
    NB_ALLOC(ux, n); NB_ALLOC(uy, n); NB_ALLOC(uz, n); NB_ALLOC(chimin, n);
    NB_ALLOC(cell_of, n); NB_ALLOC(sorted_id, n);
    NB_ALLOC(sf.ux, n); NB_ALLOC(sf.uy, n); NB_ALLOC(sf.uz, n); NB_ALLOC(sf.chimin, n); NB_ALLOC(sf.id, n);
    NB_ALLOC(counts, n); NB_ALLOC(offsets, n + 1);

    const int T = 256;
    const unsigned nblk = (unsigned)((n + T - 1) / T);
    unsigned long long *d_min = ctx->d_counters + 10;
    unsigned long long init = 0x7ff0000000000000ULL;   // +inf
    cudaError_t e = cudaMemcpyAsync(d_min, &init, sizeof(init), cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) { free(pl); return lya_cuda_fail(ctx, e, "init"); }
    { k_prep<<<nblk, T, 0, s>>>(*f, ux, uy, uz, chimin, d_min); lya_note_launch(); }
    unsigned long long min_bits = 0;
    e = cudaMemcpyAsync(&min_bits, d_min, sizeof(min_bits), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { free(pl); return lya_cuda_fail(ctx, e, "k_prep"); }
    double chi_min;
    memcpy(&chi_min, &min_bits, sizeof(double));
    if (!(chi_min < INFINITY)) { *out = pl; return LYA_OK; }       // every forest is empty

    // cell edge >= largest admissible chord (1e-9 relative margin; only has to be conservative)
    double smax = (chi_min > 0.0) ? b->rperp_max / (2.0 * chi_min) : 1.0;
    if (!(smax < 1.0)) smax = 1.0;
    double chord = 2.0 * smax * (1.0 + 1e-9) + 1e-15;
    int G = (int)floor(2.0 / chord);
    if (G > G_MAX) G = G_MAX;
    if (G < 1) G = 1;
    const int64_t n_cells = (int64_t)G * G * G;

    unsigned *hist, *cursor;
    unsigned long long *cell_start;
    NB_ALLOC(hist, n_cells); NB_ALLOC(cursor, n_cells); NB_ALLOC(cell_start, n_cells + 1);
    int64_t scan_len = (n_cells > n ? n_cells : n);
    NB_ALLOC(scan_tmp, scan_len / (SCAN_THREADS * SCAN_ITEMS) + 4);
    cudaMemsetAsync(hist, 0, sizeof(unsigned) * n_cells, s);
    cudaMemsetAsync(cursor, 0, sizeof(unsigned) * n_cells, s);

    { k_cell_hist<<<nblk, T, 0, s>>>(ux, uy, uz, chimin, n, G, cell_of, hist); lya_note_launch(); }
    e = exclusive_scan(hist, cell_start, n_cells, scan_tmp, s);
    if (e != cudaSuccess) { free(pl); return lya_cuda_fail(ctx, e, "cell scan"); }
    { k_cell_scatter<<<nblk, T, 0, s>>>(cell_of, n, cell_start, cursor, sorted_id); lya_note_launch(); }
    { k_cell_sort<<<(unsigned)((n_cells + T - 1) / T), T, 0, s>>>(cell_start, n_cells, sorted_id); lya_note_launch(); }
    unsigned long long m_ull = 0;
    e = cudaMemcpyAsync(&m_ull, cell_start + n_cells, sizeof(m_ull), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { free(pl); return lya_cuda_fail(ctx, e, "cell sort"); }
    const int64_t m = (int64_t)m_ull;                            // non-empty forests
    if (m < 2) { *out = pl; return LYA_OK; }
    { k_gather_sorted<<<(unsigned)((m + T - 1) / T), T, 0, s>>>(sorted_id, m, ux, uy, uz, chimin, sf); lya_note_launch(); }

    const unsigned wblk = (unsigned)((m * 32 + T - 1) / T);
    { k_pairs<false><<<wblk, T, 0, s>>>(sf, m, cell_start, G, b->rperp_max, counts, NULL, NULL); lya_note_launch(); }
    e = exclusive_scan(counts, offsets, m, scan_tmp, s);
    if (e != cudaSuccess) { free(pl); return lya_cuda_fail(ctx, e, "pair scan"); }
    unsigned long long total = 0;
    e = cudaMemcpyAsync(&total, offsets + m, sizeof(total), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { free(pl); return lya_cuda_fail(ctx, e, "pair count"); }
    if (total >= (1ULL << 40)) { free(pl); return lya_fail(ctx, LYA_ERR_CAPACITY, "more than 2^40 forest pairs"); }
    pl->n = (int64_t)total;
    if (total > 0) {
        e = lya_malloc(&pl->pq, sizeof(int32_t) * 2 * (size_t)total);
        if (e != cudaSuccess) { free(pl); return lya_cuda_fail(ctx, e, "lya_malloc(pair list)"); }
        { k_pairs<true><<<wblk, T, 0, s>>>(sf, m, cell_start, G, b->rperp_max, NULL, offsets, pl->pq); lya_note_launch(); }
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) { lya_free(pl->pq); free(pl); return lya_cuda_fail(ctx, e, "k_pairs<fill>"); }
    }
    *out = pl;
    *n_pairs = pl->n;
    return LYA_OK;
#undef NB_ALLOC
}
